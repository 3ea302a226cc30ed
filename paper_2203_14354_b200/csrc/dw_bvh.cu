// dw_bvh.cu -- device LBVH build (the paper names no structure, only GPU ray
// traversal [27]): triangle boxes -> scene bounds -> 63-bit Morton codes of centroids -> radix sort ->
// binary radix tree (Karras 2012) -> bottom-up refit -> subtree collapse into <= max_leaf triangle leaves ->
// compacted 64-byte traversal nodes + triangles permuted to leaf order in Moeller-Trumbore form.
#include <float.h>

#include <cub/device/device_radix_sort.cuh>
#include <cub/device/device_scan.cuh>

#include "dw_internal.cuh"

namespace {

// order-preserving float <-> uint mapping for atomicMin/Max
__device__ __forceinline__ unsigned f2o(float f) {
  unsigned u = __float_as_uint(f);
  return (u & 0x80000000u) ? ~u : (u | 0x80000000u);
}
__host__ __device__ __forceinline__ float o2f(unsigned u) {
  unsigned v = (u & 0x80000000u) ? (u & 0x7fffffffu) : ~u;
#ifdef __CUDA_ARCH__
  return __uint_as_float(v);
#else
  float f; memcpy(&f, &v, 4); return f;
#endif
}

__global__ void tri_bounds_kernel(int n, const float* __restrict__ xyz, const int32_t* __restrict__ idx,
                                  float* __restrict__ tlo, float* __restrict__ thi, unsigned* __restrict__ scene) {
  int t = blockIdx.x * blockDim.x + threadIdx.x;
  float lo[3] = {FLT_MAX, FLT_MAX, FLT_MAX}, hi[3] = {-FLT_MAX, -FLT_MAX, -FLT_MAX};
  if (t < n) {
    for (int k = 0; k < 3; ++k) {
      int v = idx[3 * (int64_t)t + k];
      for (int a = 0; a < 3; ++a) {
        float c = xyz[3 * (int64_t)v + a];
        lo[a] = fminf(lo[a], c); hi[a] = fmaxf(hi[a], c);
      }
    }
    for (int a = 0; a < 3; ++a) { tlo[3 * (int64_t)t + a] = lo[a]; thi[3 * (int64_t)t + a] = hi[a]; }
  }
  // warp reduce then one atomic per warp
  for (int a = 0; a < 3; ++a) {
    float l = lo[a], h = hi[a];
    for (int o = 16; o; o >>= 1) { l = fminf(l, __shfl_xor_sync(0xffffffffu, l, o)); h = fmaxf(h, __shfl_xor_sync(0xffffffffu, h, o)); }
    if ((threadIdx.x & 31) == 0) { atomicMin(&scene[a], f2o(l)); atomicMax(&scene[3 + a], f2o(h)); }
  }
}

__device__ __forceinline__ unsigned long long spread21(unsigned long long x) {
  x &= 0x1fffffull;
  x = (x | x << 32) & 0x1f00000000ffffull;
  x = (x | x << 16) & 0x1f0000ff0000ffull;
  x = (x | x << 8) & 0x100f00f00f00f00full;
  x = (x | x << 4) & 0x10c30c30c30c30c3ull;
  x = (x | x << 2) & 0x1249249249249249ull;
  return x;
}

__global__ void morton_kernel(int n, const float* __restrict__ tlo, const float* __restrict__ thi,
                              const unsigned* __restrict__ scene, unsigned long long* __restrict__ keys,
                              unsigned* __restrict__ vals) {
  int t = blockIdx.x * blockDim.x + threadIdx.x;
  if (t >= n) return;
  unsigned long long code = 0;
  for (int a = 0; a < 3; ++a) {
    float slo = o2f(scene[a]), shi = o2f(scene[3 + a]);
    float c = 0.5f * (tlo[3 * (int64_t)t + a] + thi[3 * (int64_t)t + a]);   // box centre
    float ext = shi - slo;
    float f = ext > 0.f ? (c - slo) / ext : 0.f;
    f = fminf(fmaxf(f, 0.f), 1.f);
    unsigned long long q = (unsigned long long)fminf(f * 2097152.f, 2097151.f);
    code |= spread21(q) << (2 - a);
  }
  keys[t] = code;
  vals[t] = (unsigned)t;
}

// ---- Karras 2012 binary radix tree over sorted keys.  Node numbering: internal i in [0, n-2], leaf j in [0, n-1]
// stored as (n - 1 + j) in the parent / box arrays.
__device__ __forceinline__ int delta(const unsigned long long* __restrict__ keys, int n, int i, int j) {
  if (j < 0 || j >= n) return -1;
  unsigned long long a = keys[i], b = keys[j];
  if (a == b) return 64 + __clz(i ^ j);
  return __clzll((long long)(a ^ b));
}

__global__ void radix_tree_kernel(int n, const unsigned long long* __restrict__ keys, int* __restrict__ left,
                                  int* __restrict__ right, int* __restrict__ parent, int* __restrict__ rfirst,
                                  int* __restrict__ rlast) {
  int i = blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= n - 1) return;
  int d = (delta(keys, n, i, i + 1) - delta(keys, n, i, i - 1)) >= 0 ? 1 : -1;
  int dmin = delta(keys, n, i, i - d);
  int lmax = 2;
  while (delta(keys, n, i, i + lmax * d) > dmin) lmax <<= 1;
  int l = 0;
  for (int t = lmax >> 1; t >= 1; t >>= 1)
    if (delta(keys, n, i, i + (l + t) * d) > dmin) l += t;
  int j = i + l * d;
  int dnode = delta(keys, n, i, j);
  int s = 0, t = l;
  do {
    t = (t + 1) >> 1;
    if (delta(keys, n, i, i + (s + t) * d) > dnode) s += t;
  } while (t > 1);
  int gamma = i + s * d + min(d, 0);
  int lo = min(i, j), hi = max(i, j);
  int L = (lo == gamma) ? (n - 1 + gamma) : gamma;
  int R = (hi == gamma + 1) ? (n - 1 + gamma + 1) : (gamma + 1);
  left[i] = L; right[i] = R;
  parent[L] = i; parent[R] = i;
  rfirst[i] = lo; rlast[i] = hi;
  if (i == 0) parent[0] = -1;
}

// bottom-up refit: second arrival at a node computes its box.  Boxes: [2n-1][6]
__global__ void refit_kernel(int n, const unsigned* __restrict__ vals, const float* __restrict__ tlo,
                             const float* __restrict__ thi, const int* __restrict__ left, const int* __restrict__ right,
                             const int* __restrict__ parent, float* __restrict__ box, int* __restrict__ flag) {
  int j = blockIdx.x * blockDim.x + threadIdx.x;
  if (j >= n) return;
  int t = vals[j];
  int me = n - 1 + j;
  for (int a = 0; a < 3; ++a) { box[6 * (int64_t)me + a] = tlo[3 * (int64_t)t + a]; box[6 * (int64_t)me + 3 + a] = thi[3 * (int64_t)t + a]; }
  __threadfence();
  int p = (n > 1) ? parent[me] : -1;
  while (p >= 0) {
    if (atomicAdd(&flag[p], 1) == 0) return;   // first arrival: the sibling subtree is not done yet
    __threadfence();
    int L = left[p], R = right[p];
    for (int a = 0; a < 3; ++a) {
      box[6 * (int64_t)p + a] = fminf(__ldcg(&box[6 * (int64_t)L + a]), __ldcg(&box[6 * (int64_t)R + a]));
      box[6 * (int64_t)p + 3 + a] = fmaxf(__ldcg(&box[6 * (int64_t)L + 3 + a]), __ldcg(&box[6 * (int64_t)R + 3 + a]));
    }
    __threadfence();
    p = parent[p];
  }
}

// statistics only: depth of the deepest leaf of the binary radix tree
__global__ void depth_kernel(int n, const int* __restrict__ parent, int* __restrict__ depth_max) {
  int j = blockIdx.x * blockDim.x + threadIdx.x;
  int depth = 0;
  if (j < n) for (int p = parent[n - 1 + j]; p >= 0; p = parent[p]) ++depth;
  for (int o = 16; o; o >>= 1) depth = max(depth, __shfl_xor_sync(0xffffffffu, depth, o));
  if ((threadIdx.x & 31) == 0) atomicMax(depth_max, depth);
}

// alive[i] = 1 for internal nodes that appear in the traversal structure: the root, and every internal node
// whose range holds more than max_leaf triangles (smaller subtrees are folded into a leaf of their parent).
__global__ void alive_kernel(int n, int max_leaf, const int* __restrict__ rfirst, const int* __restrict__ rlast,
                             int* __restrict__ alive) {
  int i = blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= n - 1) return;
  alive[i] = (i == 0 || (rlast[i] - rfirst[i] + 1) > max_leaf) ? 1 : 0;
}

__device__ __forceinline__ int child_ref(int c, int n, int max_leaf, const int* rfirst, const int* rlast, const int* newidx,
                                         int* n_leaves) {
  if (c >= n - 1) { atomicAdd(n_leaves, 1); return ~(((c - (n - 1)) << 3) | 0); }       // single-triangle leaf
  int cnt = rlast[c] - rfirst[c] + 1;
  if (cnt <= max_leaf) { atomicAdd(n_leaves, 1); return ~((rfirst[c] << 3) | (cnt - 1)); }
  return newidx[c];
}

__global__ void emit_nodes_kernel(int n, int max_leaf, const int* __restrict__ left, const int* __restrict__ right,
                                  const int* __restrict__ rfirst, const int* __restrict__ rlast,
                                  const int* __restrict__ alive, const int* __restrict__ newidx,
                                  const float* __restrict__ box, float4* __restrict__ nodes, int* __restrict__ n_leaves) {
  int i = blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= n - 1 || !alive[i]) return;
  int L = left[i], R = right[i];
  const float* b0 = box + 6 * (int64_t)L;
  const float* b1 = box + 6 * (int64_t)R;
  int r0 = child_ref(L, n, max_leaf, rfirst, rlast, newidx, n_leaves);
  int r1 = child_ref(R, n, max_leaf, rfirst, rlast, newidx, n_leaves);
  float4* o = nodes + 4 * (int64_t)newidx[i];
  o[0] = make_float4(b0[0], b0[1], b0[2], b0[3]);
  o[1] = make_float4(b0[4], b0[5], b1[0], b1[1]);
  o[2] = make_float4(b1[2], b1[3], b1[4], b1[5]);
  o[3] = make_float4(__int_as_float(r0), __int_as_float(r1), 0.f, 0.f);
}

// n == 1: a root whose first child is the only triangle and whose second child is empty
__global__ void emit_single_kernel(const float* __restrict__ tlo, const float* __restrict__ thi, float4* __restrict__ nodes) {
  nodes[0] = make_float4(tlo[0], tlo[1], tlo[2], thi[0]);
  nodes[1] = make_float4(thi[1], thi[2], FLT_MAX, FLT_MAX);
  nodes[2] = make_float4(FLT_MAX, -FLT_MAX, -FLT_MAX, -FLT_MAX);
  nodes[3] = make_float4(__int_as_float(~0), __int_as_float(DW_REF_NONE), 0.f, 0.f);
}

__global__ void pack_tris_kernel(int n, const unsigned* __restrict__ vals, const float* __restrict__ xyz,
                                 const int32_t* __restrict__ idx, const uint32_t* __restrict__ code,
                                 const int32_t* __restrict__ chan, float4* __restrict__ tris) {
  int j = blockIdx.x * blockDim.x + threadIdx.x;
  if (j >= n) return;
  int t = vals[j];
  int i0 = idx[3 * (int64_t)t], i1 = idx[3 * (int64_t)t + 1], i2 = idx[3 * (int64_t)t + 2];
  float v0[3], e1[3], e2[3];
  for (int a = 0; a < 3; ++a) {
    v0[a] = xyz[3 * (int64_t)i0 + a];
    e1[a] = xyz[3 * (int64_t)i1 + a] - v0[a];
    e2[a] = xyz[3 * (int64_t)i2 + a] - v0[a];
  }
  float4* o = tris + 3 * (int64_t)j;
  o[0] = make_float4(v0[0], v0[1], v0[2], e1[0]);
  o[1] = make_float4(e1[1], e1[2], e2[0], e2[1]);
  o[2] = make_float4(e2[2], __int_as_float(t), __uint_as_float(code[t]), __int_as_float(chan[t]));
}

}  // namespace

#define DW_B(call) do { cudaError_t e__ = (call); if (e__ != cudaSuccess) { rc = dw_fail(c, DW_E_CUDA, "%s failed: %s (%s:%d)", \
    #call, cudaGetErrorString(e__), __FILE__, __LINE__); goto done; } } while (0)

int dw_bvh_build_impl(dw_ctx* c, const dw_build_params* params, dw_build_stats* stats, cudaStream_t stream) {
  int rc = DW_OK;
  const int n = (int)c->n_tri;
  int max_leaf = (params && params->max_leaf_tris) ? params->max_leaf_tris : 4;
  if (max_leaf < 1 || max_leaf > 8) return dw_fail(c, DW_E_ARG, "dw_build_bvh: max_leaf_tris must be in 1..8");
  cudaFree(c->d_nodes); cudaFree(c->d_tris);
  c->d_nodes = nullptr; c->d_tris = nullptr; c->built = false;
  if (stats) memset(stats, 0, sizeof *stats);

  float *tlo = nullptr, *thi = nullptr, *box = nullptr;
  unsigned *scene = nullptr, *vals = nullptr, *vals2 = nullptr;
  unsigned long long *keys = nullptr, *keys2 = nullptr;
  int *left = nullptr, *right = nullptr, *parent = nullptr, *rfirst = nullptr, *rlast = nullptr, *flag = nullptr,
      *alive = nullptr, *newidx = nullptr, *misc = nullptr;
  void* tmp = nullptr;
  size_t tmp_bytes = 0, tmp2 = 0;
  cudaEvent_t ev0 = nullptr, ev1 = nullptr;
  unsigned h_scene[6];
  int h_misc[4] = {0, 0, 0, 0};
  int n_nodes = 1;
  const int B = 256;
  const unsigned G = (unsigned)((std::max(n, 1) + B - 1) / B);

  if (n == 0) {   // empty world: one node with two empty children
    float4 h[4] = {make_float4(FLT_MAX, FLT_MAX, FLT_MAX, -FLT_MAX), make_float4(-FLT_MAX, -FLT_MAX, FLT_MAX, FLT_MAX),
                   make_float4(FLT_MAX, -FLT_MAX, -FLT_MAX, -FLT_MAX), make_float4(0, 0, 0, 0)};
    int none = DW_REF_NONE;
    memcpy(&h[3].x, &none, 4); memcpy(&h[3].y, &none, 4);
    DW_B(cudaMalloc(&c->d_nodes, sizeof h));
    DW_B(cudaMalloc(&c->d_tris, 48));
    DW_B(cudaMemcpy(c->d_nodes, h, sizeof h, cudaMemcpyHostToDevice));
    c->bvh = DwBvh{c->d_nodes, c->d_tris, 1, 0, 0.f};
    c->built = true;
    return DW_OK;
  }

  DW_B(cudaEventCreate(&ev0)); DW_B(cudaEventCreate(&ev1));
  DW_B(cudaMalloc(&tlo, sizeof(float) * 3 * n)); DW_B(cudaMalloc(&thi, sizeof(float) * 3 * n));
  DW_B(cudaMalloc(&box, sizeof(float) * 6 * (2 * (size_t)n)));
  DW_B(cudaMalloc(&scene, sizeof(unsigned) * 6));
  DW_B(cudaMalloc(&keys, 8 * (size_t)n)); DW_B(cudaMalloc(&keys2, 8 * (size_t)n));
  DW_B(cudaMalloc(&vals, 4 * (size_t)n)); DW_B(cudaMalloc(&vals2, 4 * (size_t)n));
  DW_B(cudaMalloc(&left, 4 * (size_t)n)); DW_B(cudaMalloc(&right, 4 * (size_t)n));
  DW_B(cudaMalloc(&parent, 4 * (2 * (size_t)n))); DW_B(cudaMalloc(&rfirst, 4 * (size_t)n)); DW_B(cudaMalloc(&rlast, 4 * (size_t)n));
  DW_B(cudaMalloc(&flag, 4 * (size_t)n)); DW_B(cudaMalloc(&alive, 4 * (size_t)n)); DW_B(cudaMalloc(&newidx, 4 * (size_t)n));
  DW_B(cudaMalloc(&misc, 16));
  DW_B(cub::DeviceRadixSort::SortPairs(nullptr, tmp_bytes, keys, keys2, vals, vals2, n, 0, 63, stream));
  DW_B(cub::DeviceScan::ExclusiveSum(nullptr, tmp2, alive, newidx, std::max(n - 1, 1), stream));
  tmp_bytes = std::max(tmp_bytes, tmp2);
  DW_B(cudaMalloc(&tmp, tmp_bytes));

  DW_B(cudaEventRecord(ev0, stream));
  {
    unsigned init[6] = {0xffffffffu, 0xffffffffu, 0xffffffffu, 0u, 0u, 0u};
    DW_B(cudaMemcpyAsync(scene, init, sizeof init, cudaMemcpyHostToDevice, stream));
  }
  DW_B(cudaMemsetAsync(flag, 0, 4 * (size_t)n, stream));
  DW_B(cudaMemsetAsync(misc, 0, 16, stream));
  tri_bounds_kernel<<<G, B, 0, stream>>>(n, c->d_xyz, c->d_idx, tlo, thi, scene);
  morton_kernel<<<G, B, 0, stream>>>(n, tlo, thi, scene, keys, vals);
  DW_B(cub::DeviceRadixSort::SortPairs(tmp, tmp_bytes, keys, keys2, vals, vals2, n, 0, 63, stream));
  DW_B(cudaMalloc(&c->d_tris, 48 * (size_t)n));
  pack_tris_kernel<<<G, B, 0, stream>>>(n, vals2, c->d_xyz, c->d_idx, c->d_code, c->d_chan, c->d_tris);
  if (n >= 2) {
    radix_tree_kernel<<<G, B, 0, stream>>>(n, keys2, left, right, parent, rfirst, rlast);
    refit_kernel<<<G, B, 0, stream>>>(n, vals2, tlo, thi, left, right, parent, box, flag);
    depth_kernel<<<G, B, 0, stream>>>(n, parent, misc + 0);
    alive_kernel<<<G, B, 0, stream>>>(n, max_leaf, rfirst, rlast, alive);
    DW_B(cub::DeviceScan::ExclusiveSum(tmp, tmp_bytes, alive, newidx, n - 1, stream));
    // number of alive nodes = newidx[n-2] + alive[n-2]
    int h_last[2];
    DW_B(cudaMemcpyAsync(&h_last[0], newidx + (n - 2), 4, cudaMemcpyDeviceToHost, stream));
    DW_B(cudaMemcpyAsync(&h_last[1], alive + (n - 2), 4, cudaMemcpyDeviceToHost, stream));
    DW_B(cudaStreamSynchronize(stream));
    n_nodes = h_last[0] + h_last[1];
    DW_B(cudaMalloc(&c->d_nodes, 64 * (size_t)n_nodes));
    emit_nodes_kernel<<<G, B, 0, stream>>>(n, max_leaf, left, right, rfirst, rlast, alive, newidx, box, c->d_nodes, misc + 1);
  } else {
    DW_B(cudaMalloc(&c->d_nodes, 64));
    emit_single_kernel<<<1, 1, 0, stream>>>(tlo, thi, c->d_nodes);
    h_misc[0] = 1; h_misc[1] = 1;
  }
  DW_B(cudaGetLastError());
  DW_B(cudaEventRecord(ev1, stream));
  DW_B(cudaMemcpyAsync(h_scene, scene, sizeof h_scene, cudaMemcpyDeviceToHost, stream));
  if (n >= 2) DW_B(cudaMemcpyAsync(h_misc, misc, 8, cudaMemcpyDeviceToHost, stream));
  DW_B(cudaStreamSynchronize(stream));
  {
    float mx = 0.f;
    float lo[3], hi[3];
    for (int a = 0; a < 3; ++a) { lo[a] = o2f(h_scene[a]); hi[a] = o2f(h_scene[3 + a]); mx = fmaxf(mx, fmaxf(fabsf(lo[a]), fabsf(hi[a]))); }
    // Length tolerance: a few fp32 spacings of the largest coordinate (positions cannot be resolved finer).
    float eps_len = 4.0f * 1.1920929e-7f * mx;
    c->bvh = DwBvh{c->d_nodes, c->d_tris, n_nodes, n, eps_len};
    c->built = true;
    if (stats) {
      stats->n_tri = n; stats->n_nodes = n_nodes; stats->node_bytes = 64ll * n_nodes; stats->tri_bytes = 48ll * n;
      stats->max_depth = h_misc[0]; stats->n_leaves = h_misc[1];
      for (int a = 0; a < 3; ++a) { stats->scene_lo[a] = lo[a]; stats->scene_hi[a] = hi[a]; }
      cudaEventElapsedTime(&stats->build_ms, ev0, ev1);
    }
  }
done:
  cudaFree(tlo); cudaFree(thi); cudaFree(box); cudaFree(scene); cudaFree(keys); cudaFree(keys2); cudaFree(vals);
  cudaFree(vals2); cudaFree(left); cudaFree(right); cudaFree(parent); cudaFree(rfirst); cudaFree(rlast); cudaFree(flag);
  cudaFree(alive); cudaFree(newidx); cudaFree(misc); cudaFree(tmp);
  if (ev0) cudaEventDestroy(ev0);
  if (ev1) cudaEventDestroy(ev1);
  if (rc != DW_OK) { cudaFree(c->d_nodes); cudaFree(c->d_tris); c->d_nodes = nullptr; c->d_tris = nullptr; c->built = false; }
  return rc;
}
