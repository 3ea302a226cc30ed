// dw_bvh.cu -- device BVH build (the paper names no structure, only GPU ray traversal [27],
// P:111): triangle boxes -> scene bounds -> 63-bit Morton codes of box centres -> radix sort -> bottom-up binary tree by
// parallel locally-ordered clustering over the Morton order (PLOC, Meister & Bittner 2018: every cluster looks
// +-radius positions around itself for the partner that gives the smallest merged box; mutual choices merge) ->
// depth-first triangle order, subtrees of <= max_leaf triangles folded into leaves -> greedy collapse into 4-wide
// nodes (open the child of largest area first) -> 128-byte SoA traversal nodes + Moeller-Trumbore triangle records.
// Why PLOC and 4-wide: DESIGN.md section 5 (node visits and box tests per query against the Morton radix tree).
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

// ---- triangle references.  A triangle whose box is longer than smax = (largest scene extent) / split_div is represented by
// several references, each with the tight box of the part of the triangle inside a sub-box (clip, bound, halve the longest
// axis, repeat): the long slivers of fans and the tall wall panels otherwise give leaf boxes that overlap over metres and
// most triangle tests are misses (profiles/r01_propagate_bvh4_c2.md, capture 5).  A reference is only a box: leaves hold
// the whole triangle, so a triangle can be tested twice by one ray, which the first-hit rule (nearest, then lowest id)
// does not notice.  The union of the boxes of a triangle covers it; boxes are padded by `pad`.
constexpr int kClipMax = 10;      // a triangle clipped by an axis-aligned box has at most 9 vertices
constexpr int kSplitStack = 24;

// Sutherland-Hodgman against one axis plane: keep coordinate[axis] >= val (keep_ge) or <= val.
__device__ int clip_axis(const float (*in)[3], int n, int axis, float val, bool keep_ge, float (*out)[3]) {
  int m = 0;
  for (int i = 0; i < n; ++i) {
    const float* a = in[i];
    const float* b = in[(i + 1 == n) ? 0 : i + 1];
    const bool ia = keep_ge ? a[axis] >= val : a[axis] <= val;
    const bool ib = keep_ge ? b[axis] >= val : b[axis] <= val;
    if (ia && m < kClipMax) { out[m][0] = a[0]; out[m][1] = a[1]; out[m][2] = a[2]; ++m; }
    if (ia != ib && m < kClipMax) {
      const float w = (val - a[axis]) / (b[axis] - a[axis]);
      for (int c = 0; c < 3; ++c) out[m][c] = fmaf(w, b[c] - a[c], a[c]);
      out[m][axis] = val;
      ++m;
    }
  }
  return m;
}

// References of one triangle.  out_lo / out_hi == nullptr: count only.  Returns the number of references.  cap > 0: room for
// cap boxes; pieces beyond it are merged into the last box (the refit must fill exactly as many references as the tree has).
__device__ int split_triangle(const float v[3][3], const float tlo[3], const float thi[3], float smax, float pad,
                              float* out_lo, float* out_hi, int cap = 0) {
  float ext = fmaxf(thi[0] - tlo[0], fmaxf(thi[1] - tlo[1], thi[2] - tlo[2]));
  if (!(ext > smax)) {
    if (out_lo) for (int c = 0; c < 3; ++c) { out_lo[c] = tlo[c]; out_hi[c] = thi[c]; }
    return 1;
  }
  float slo[kSplitStack][3], shi[kSplitStack][3];
  float pa[kClipMax][3], pb[kClipMax][3];
  int sp = 0, cnt = 0;
  for (int c = 0; c < 3; ++c) { slo[0][c] = tlo[c]; shi[0][c] = thi[c]; }
  sp = 1;
  for (int iter = 0; iter < 8192 && sp > 0; ++iter) {
    --sp;
    float blo[3] = {slo[sp][0], slo[sp][1], slo[sp][2]}, bhi[3] = {shi[sp][0], shi[sp][1], shi[sp][2]};
    int np = 3;
    for (int i = 0; i < 3; ++i) for (int c = 0; c < 3; ++c) pa[i][c] = v[i][c];
    for (int axis = 0; axis < 3 && np > 0; ++axis) {
      np = clip_axis(pa, np, axis, blo[axis], true, pb);
      if (np > 0) np = clip_axis(pb, np, axis, bhi[axis], false, pa);
    }
    if (np == 0) continue;                                       // this sub-box holds nothing of the triangle
    float lo[3] = {FLT_MAX, FLT_MAX, FLT_MAX}, hi[3] = {-FLT_MAX, -FLT_MAX, -FLT_MAX};
    for (int i = 0; i < np; ++i) for (int c = 0; c < 3; ++c) { lo[c] = fminf(lo[c], pa[i][c]); hi[c] = fmaxf(hi[c], pa[i][c]); }
    for (int c = 0; c < 3; ++c) { lo[c] = fmaxf(lo[c], blo[c]); hi[c] = fminf(hi[c], bhi[c]); }
    int ax = 0;
    float e = hi[0] - lo[0];
    if (hi[1] - lo[1] > e) { e = hi[1] - lo[1]; ax = 1; }
    if (hi[2] - lo[2] > e) { e = hi[2] - lo[2]; ax = 2; }
    if (e <= smax || sp + 2 > kSplitStack) {
      if (out_lo) {
        if (cap > 0 && cnt >= cap) {
          for (int c = 0; c < 3; ++c) {
            out_lo[3 * (cap - 1) + c] = fminf(out_lo[3 * (cap - 1) + c], lo[c] - pad);
            out_hi[3 * (cap - 1) + c] = fmaxf(out_hi[3 * (cap - 1) + c], hi[c] + pad);
          }
        } else {
          for (int c = 0; c < 3; ++c) { out_lo[3 * cnt + c] = lo[c] - pad; out_hi[3 * cnt + c] = hi[c] + pad; }
        }
      }
      ++cnt;
      continue;
    }
    const float mid = 0.5f * (lo[ax] + hi[ax]);
    for (int c = 0; c < 3; ++c) { slo[sp][c] = lo[c]; shi[sp][c] = hi[c]; slo[sp + 1][c] = lo[c]; shi[sp + 1][c] = hi[c]; }
    shi[sp][ax] = mid; slo[sp + 1][ax] = mid;
    sp += 2;
  }
  if (cnt == 0) {                                                // rounding clipped everything away: one reference, the whole box
    if (out_lo) for (int c = 0; c < 3; ++c) { out_lo[c] = tlo[c] - pad; out_hi[c] = thi[c] + pad; }
    cnt = 1;
  }
  return cnt;
}

__device__ __forceinline__ void load_tri(const float* __restrict__ xyz, const int32_t* __restrict__ idx, int t, float v[3][3]) {
  for (int k = 0; k < 3; ++k) {
    const int vi = idx[3 * (int64_t)t + k];
    for (int c = 0; c < 3; ++c) v[k][c] = xyz[3 * (int64_t)vi + c];
  }
}
__device__ __forceinline__ float split_smax(const unsigned* __restrict__ scene, int split_div) {
  if (split_div <= 0) return FLT_MAX;
  const float e = fmaxf(o2f(scene[3]) - o2f(scene[0]), fmaxf(o2f(scene[4]) - o2f(scene[1]), o2f(scene[5]) - o2f(scene[2])));
  return e / (float)split_div;
}
__global__ void split_count_kernel(int n, const float* __restrict__ xyz, const int32_t* __restrict__ idx,
                                   const float* __restrict__ tlo, const float* __restrict__ thi,
                                   const unsigned* __restrict__ scene, int split_div, int* __restrict__ counts) {
  int t = blockIdx.x * blockDim.x + threadIdx.x;
  if (t >= n) return;
  float v[3][3];
  load_tri(xyz, idx, t, v);
  counts[t] = split_triangle(v, tlo + 3 * (int64_t)t, thi + 3 * (int64_t)t, split_smax(scene, split_div), 0.f, nullptr, nullptr);
}
__global__ void split_emit_kernel(int n, const float* __restrict__ xyz, const int32_t* __restrict__ idx,
                                  const float* __restrict__ tlo, const float* __restrict__ thi,
                                  const unsigned* __restrict__ scene, int split_div, float pad, const int* __restrict__ offs,
                                  const int* __restrict__ counts, float* __restrict__ rlo, float* __restrict__ rhi,
                                  int* __restrict__ ref_tri) {
  int t = blockIdx.x * blockDim.x + threadIdx.x;
  if (t >= n) return;
  float v[3][3];
  load_tri(xyz, idx, t, v);
  const int o = offs[t], cnt = counts[t];
  const int made = split_triangle(v, tlo + 3 * (int64_t)t, thi + 3 * (int64_t)t, split_smax(scene, split_div), cnt > 1 ? pad : 0.f,
                                  rlo + 3 * (int64_t)o, rhi + 3 * (int64_t)o);
  for (int k = 0; k < cnt; ++k) {
    ref_tri[o + k] = t;
    if (k >= made)                                               // cannot happen (same arithmetic as the count pass); keep the box valid
      for (int c = 0; c < 3; ++c) { rlo[3 * (int64_t)(o + k) + c] = tlo[3 * (int64_t)t + c]; rhi[3 * (int64_t)(o + k) + c] = thi[3 * (int64_t)t + c]; }
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

// ---- binary tree.  Node numbering: leaf j in [0, n-1] = the j-th triangle in Morton order; internal nodes n .. 2n-2 in
// the order PLOC creates them (children always before parents), so the root is node 2n-2.  Boxes: blo/bhi[node].xyz.
__device__ __forceinline__ float half_area(float4 lo, float4 hi) {
  float ex = hi.x - lo.x, ey = hi.y - lo.y, ez = hi.z - lo.z;
  return fmaf(ex, ey, fmaf(ey, ez, ex * ez));
}
__device__ __forceinline__ float4 min4(float4 a, float4 b) { return make_float4(fminf(a.x, b.x), fminf(a.y, b.y), fminf(a.z, b.z), 0.f); }
__device__ __forceinline__ float4 max4(float4 a, float4 b) { return make_float4(fmaxf(a.x, b.x), fmaxf(a.y, b.y), fmaxf(a.z, b.z), 0.f); }

__global__ void ploc_init_kernel(int n, const unsigned* __restrict__ vals, const float* __restrict__ tlo,
                                 const float* __restrict__ thi, float4* __restrict__ blo, float4* __restrict__ bhi,
                                 int* __restrict__ cnode, float4* __restrict__ clo, float4* __restrict__ chi,
                                 int* __restrict__ size, int* __restrict__ parent, int* __restrict__ leftmost) {
  int j = blockIdx.x * blockDim.x + threadIdx.x;
  if (j >= n) return;
  int t = vals[j];
  float4 lo = make_float4(tlo[3 * (int64_t)t], tlo[3 * (int64_t)t + 1], tlo[3 * (int64_t)t + 2], 0.f);
  float4 hi = make_float4(thi[3 * (int64_t)t], thi[3 * (int64_t)t + 1], thi[3 * (int64_t)t + 2], 0.f);
  blo[j] = lo; bhi[j] = hi; clo[j] = lo; chi[j] = hi;
  cnode[j] = j; size[j] = 1; parent[j] = -1; leftmost[j] = j;
}

// Nearest neighbour of cluster i among positions i-radius .. i+radius: smallest merged half-area, ties -> smallest
// position.  The pair that is smallest in (area, i, j) order always chooses each other, so every round merges.
__global__ void ploc_nn_kernel(int m, int radius, const float4* __restrict__ clo, const float4* __restrict__ chi,
                               int* __restrict__ nn) {
  int i = blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= m) return;
  float4 lo = clo[i], hi = chi[i];
  float best = FLT_MAX;
  int bj = -1;
  int j0 = max(i - radius, 0), j1 = min(i + radius, m - 1);
  for (int j = j0; j <= j1; ++j) {
    if (j == i) continue;
    float a = half_area(min4(lo, clo[j]), max4(hi, chi[j]));
    if (a < best || bj < 0) { best = a; bj = j; }          // strict <: the first (smallest) position wins ties
  }
  nn[i] = bj;
}

// The rounds run without the host: the number of clusters m and the next node index `base` live on the device, in two copies
// that the rounds use alternately (st[0..1] for even rounds, st[2..3] for odd ones; st[4] counts the rounds, st[5] is an error
// flag).  Every kernel of a round is launched over the n positions of the first round and returns where i >= m; the host reads m
// back once per chunk of rounds.  (Round 1: two CUB scans and an 8-byte read-back per round, 55-70 rounds: the build was latency.)
// keep = 0 for the higher position of a mutual pair (it disappears); isnew = 1 for the lower one (a node is made).  flag bit 0 keep,
// bit 1 isnew.  bsum[block] = (kept, new) of the block's positions.
__global__ void ploc_nn_kernel_dev(const int* __restrict__ st, int radius, const float4* __restrict__ clo, const float4* __restrict__ chi,
                                   int* __restrict__ nn) {
  const int m = st[0];
  int i = blockIdx.x * blockDim.x + threadIdx.x;
  if (m <= 1 || i >= m) return;
  float4 lo = clo[i], hi = chi[i];
  float best = FLT_MAX;
  int bj = -1;
  int j0 = max(i - radius, 0), j1 = min(i + radius, m - 1);
  for (int j = j0; j <= j1; ++j) {
    if (j == i) continue;
    float a = half_area(min4(lo, clo[j]), max4(hi, chi[j]));
    if (a < best || bj < 0) { best = a; bj = j; }          // strict <: the first (smallest) position wins ties
  }
  nn[i] = bj;
}
__device__ __forceinline__ int2 block_excl_scan2(int2 v, int2* total) {   // exclusive scan of two counters over a 256-thread block
  __shared__ int2 wsum[8];
  const int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
  int2 inc = v;
  for (int o = 1; o < 32; o <<= 1) {
    const int ux = __shfl_up_sync(0xffffffffu, inc.x, o), uy = __shfl_up_sync(0xffffffffu, inc.y, o);
    if (lane >= o) { inc.x += ux; inc.y += uy; }
  }
  if (lane == 31) wsum[w] = inc;
  __syncthreads();
  int2 off = make_int2(0, 0), tot = make_int2(0, 0);
  for (int k = 0; k < 8; ++k) { if (k < w) { off.x += wsum[k].x; off.y += wsum[k].y; } tot.x += wsum[k].x; tot.y += wsum[k].y; }
  __syncthreads();
  if (total) *total = tot;
  return make_int2(off.x + inc.x - v.x, off.y + inc.y - v.y);
}
__global__ void __launch_bounds__(256) ploc_mark_kernel_dev(const int* __restrict__ st, const int* __restrict__ nn, unsigned char* __restrict__ flag,
                                                            int2* __restrict__ bsum) {
  const int m = st[0];
  if (m <= 1 || (int)(blockIdx.x * blockDim.x) >= m) return;
  int i = blockIdx.x * blockDim.x + threadIdx.x;
  int keep = 0, isnew = 0;
  if (i < m) {
    int j = nn[i];
    bool mutual = j >= 0 && nn[j] == i;
    keep = (mutual && i > j) ? 0 : 1;
    isnew = (mutual && i < j) ? 1 : 0;
    flag[i] = (unsigned char)(keep | (isnew << 1));
  }
  int2 tot;
  block_excl_scan2(make_int2(keep, isnew), &tot);
  if (threadIdx.x == 0) bsum[blockIdx.x] = tot;
}
// one block: exclusive scan of the block sums, and the state of the next round
__global__ void __launch_bounds__(1024) ploc_scan_kernel_dev(const int* __restrict__ st, int* __restrict__ st_next, int* __restrict__ st_common,
                                                             const int2* __restrict__ bsum, int2* __restrict__ boff) {
  const int m = st[0], base = st[1];
  if (m <= 1) { if (threadIdx.x == 0) { st_next[0] = m; st_next[1] = base; } return; }
  const int nb = (m + 255) / 256;
  __shared__ int2 wsum[32];
  __shared__ int2 carry;
  if (threadIdx.x == 0) carry = make_int2(0, 0);
  __syncthreads();
  const int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
  for (int b0 = 0; b0 < nb; b0 += 1024) {
    const int b = b0 + threadIdx.x;
    const int2 v = b < nb ? bsum[b] : make_int2(0, 0);
    int2 inc = v;
    for (int o = 1; o < 32; o <<= 1) {
      const int ux = __shfl_up_sync(0xffffffffu, inc.x, o), uy = __shfl_up_sync(0xffffffffu, inc.y, o);
      if (lane >= o) { inc.x += ux; inc.y += uy; }
    }
    if (lane == 31) wsum[w] = inc;
    __syncthreads();
    int2 off = carry;
    int2 tot = make_int2(0, 0);
    for (int k = 0; k < 32; ++k) { if (k < w) { off.x += wsum[k].x; off.y += wsum[k].y; } tot.x += wsum[k].x; tot.y += wsum[k].y; }
    if (b < nb) boff[b] = make_int2(off.x + inc.x - v.x, off.y + inc.y - v.y);
    __syncthreads();
    if (threadIdx.x == 0) { carry.x += tot.x; carry.y += tot.y; }
    __syncthreads();
  }
  if (threadIdx.x == 0) {
    const int m_new = carry.x;
    if (m_new >= m || m_new < 1 || m - m_new != carry.y) st_common[1] = 1;      // a round always merges at least one pair
    st_next[0] = m_new; st_next[1] = base + (m - m_new);
    st_common[0] += 1;
  }
}
__global__ void __launch_bounds__(256) ploc_apply_kernel_dev(const int* __restrict__ st, const int* __restrict__ nn, const unsigned char* __restrict__ flag,
                                                             const int2* __restrict__ boff, const int* __restrict__ cnode_in,
                                                             const float4* __restrict__ clo_in, const float4* __restrict__ chi_in,
                                                             int* __restrict__ cnode_out, float4* __restrict__ clo_out, float4* __restrict__ chi_out,
                                                             int* __restrict__ left, int* __restrict__ right, int* __restrict__ parent,
                                                             float4* __restrict__ blo, float4* __restrict__ bhi, int* __restrict__ size) {
  const int m = st[0], base = st[1];
  if (m <= 1 || (int)(blockIdx.x * blockDim.x) >= m) return;
  int i = blockIdx.x * blockDim.x + threadIdx.x;
  const int f = i < m ? flag[i] : 0;
  const int keep = f & 1, isnew = (f >> 1) & 1;
  const int2 loc = block_excl_scan2(make_int2(keep, isnew), nullptr);
  if (i >= m || !keep) return;
  const int2 bo = boff[blockIdx.x];
  const int pos = bo.x + loc.x;
  if (isnew) {
    int j = nn[i];
    int node = base + bo.y + loc.y;
    int a = cnode_in[i], b = cnode_in[j];
    float4 lo = min4(clo_in[i], clo_in[j]), hi = max4(chi_in[i], chi_in[j]);
    left[node] = a; right[node] = b; parent[a] = node; parent[b] = node; parent[node] = -1;
    blo[node] = lo; bhi[node] = hi;
    size[node] = size[a] + size[b];
    cnode_out[pos] = node; clo_out[pos] = lo; chi_out[pos] = hi;
  } else {
    cnode_out[pos] = cnode_in[i]; clo_out[pos] = clo_in[i]; chi_out[pos] = chi_in[i];
  }
}

// Depth-first slot of every triangle: walking from leaf j to the root, every time the walk arrives from a right child
// the whole left sibling subtree lies before j.  While the walk has only taken left-child steps, j is the leftmost
// leaf of the node reached (leftmost[] gives a leaf group its first slot later).
__global__ void leaf_walk_kernel(int n, const int* __restrict__ left, const int* __restrict__ parent,
                                 const int* __restrict__ size, int* __restrict__ slot, int* __restrict__ leftmost,
                                 int* __restrict__ depth_max) {
  int j = blockIdx.x * blockDim.x + threadIdx.x;
  int depth = 0;
  if (j < n) {
    int off = 0, cur = j;
    bool all_left = true;
    for (int p = parent[cur]; p >= 0; p = parent[cur]) {
      int l = left[p];
      if (l != cur) { off += size[l]; all_left = false; }
      else if (all_left) leftmost[p] = j;
      cur = p;
      ++depth;
    }
    slot[j] = off;
  }
  for (int o = 16; o; o >>= 1) depth = max(depth, __shfl_xor_sync(0xffffffffu, depth, o));
  if ((threadIdx.x & 31) == 0) atomicMax(depth_max, depth);
}

struct WideTask { int bnode, widx; };

__device__ __forceinline__ void write_wide(float4* __restrict__ nodes, int w, const float4* lo, const float4* hi, const int* ref) {
  float4* o = nodes + 8 * (int64_t)w;
  o[0] = make_float4(lo[0].x, lo[1].x, lo[2].x, lo[3].x);
  o[1] = make_float4(lo[0].y, lo[1].y, lo[2].y, lo[3].y);
  o[2] = make_float4(lo[0].z, lo[1].z, lo[2].z, lo[3].z);
  o[3] = make_float4(hi[0].x, hi[1].x, hi[2].x, hi[3].x);
  o[4] = make_float4(hi[0].y, hi[1].y, hi[2].y, hi[3].y);
  o[5] = make_float4(hi[0].z, hi[1].z, hi[2].z, hi[3].z);
  o[6] = make_float4(__int_as_float(ref[0]), __int_as_float(ref[1]), __int_as_float(ref[2]), __int_as_float(ref[3]));
  o[7] = make_float4(0.f, 0.f, 0.f, 0.f);
}

// One level of the collapse: binary node b (more than max_leaf triangles) becomes wide node w.  Its two children are
// opened greedily, largest box first, until four remain or none can be opened (a subtree of <= max_leaf triangles is a
// leaf and stays closed).  Children that are still subtrees get a wide index and a task for the next level.
// The level's task count is read from the device (lvl[level]; the children made here are counted in lvl[level + 1]), so that the
// levels follow each other without the host: it launches one kernel per possible level and reads the counts back once.
__global__ void wide_collapse_kernel(const int* __restrict__ lvl_in, int* __restrict__ lvl_out, const WideTask* __restrict__ tasks,
                                     WideTask* __restrict__ next,
                                     int* __restrict__ counters /* [1] wide nodes, [2] leaves */,
                                     int max_leaf, const int* __restrict__ left, const int* __restrict__ right,
                                     const int* __restrict__ size, const float4* __restrict__ blo,
                                     const float4* __restrict__ bhi, const int* __restrict__ slot,
                                     const int* __restrict__ leftmost, float4* __restrict__ nodes) {
  const int n_tasks = *lvl_in;
  for (int i = blockIdx.x * blockDim.x + threadIdx.x; i < n_tasks; i += gridDim.x * blockDim.x) {
  const int b = tasks[i].bnode, w = tasks[i].widx;
  int kid[4];
  int nk = 2;
  kid[0] = left[b]; kid[1] = right[b];
  while (nk < 4) {
    int pick = -1;
    float amax = -1.f;
    for (int k = 0; k < nk; ++k) {
      if (size[kid[k]] <= max_leaf) continue;
      float a = half_area(blo[kid[k]], bhi[kid[k]]);
      if (a > amax) { amax = a; pick = k; }
    }
    if (pick < 0) break;
    int c = kid[pick];
    kid[pick] = left[c];
    kid[nk++] = right[c];
  }
  float4 lo[4], hi[4];
  int ref[4];
  for (int k = 0; k < 4; ++k) {
    lo[k] = make_float4(FLT_MAX, FLT_MAX, FLT_MAX, 0.f); hi[k] = make_float4(-FLT_MAX, -FLT_MAX, -FLT_MAX, 0.f); ref[k] = DW_REF_NONE;
    if (k >= nk) continue;
    int c = kid[k];
    lo[k] = blo[c]; hi[k] = bhi[c];
    if (size[c] <= max_leaf) {
      ref[k] = ~((slot[leftmost[c]] << 3) | (size[c] - 1));
      atomicAdd(&counters[2], 1);
    } else {
      int widx = atomicAdd(&counters[1], 1);
      ref[k] = widx;
      next[atomicAdd(lvl_out, 1)] = WideTask{c, widx};
    }
  }
  write_wide(nodes, w, lo, hi, ref);
  }
}

// A world of <= max_leaf triangles (or none): one wide node whose first child is the only leaf (or nothing).
__global__ void wide_single_kernel(int n, const float4* __restrict__ blo, const float4* __restrict__ bhi, float4* __restrict__ nodes) {
  float4 lo[4], hi[4];
  int ref[4];
  for (int k = 0; k < 4; ++k) { lo[k] = make_float4(FLT_MAX, FLT_MAX, FLT_MAX, 0.f); hi[k] = make_float4(-FLT_MAX, -FLT_MAX, -FLT_MAX, 0.f); ref[k] = DW_REF_NONE; }
  if (n > 0) { lo[0] = blo[2 * n - 2]; hi[0] = bhi[2 * n - 2]; ref[0] = ~((0 << 3) | (n - 1)); }
  write_wide(nodes, 0, lo, hi, ref);
}

// triangle j of the Morton order goes to depth-first slot[j]
__global__ void pack_tris_kernel(int n, const unsigned* __restrict__ vals, const int* __restrict__ ref_tri, const int* __restrict__ slot,
                                 const float* __restrict__ xyz, const int32_t* __restrict__ idx,
                                 const uint32_t* __restrict__ code, const int32_t* __restrict__ chan,
                                 float4* __restrict__ tris, int* __restrict__ slot_ref) {
  int j = blockIdx.x * blockDim.x + threadIdx.x;
  if (j >= n) return;
  int t = ref_tri[vals[j]];                  // reference -> triangle (several references may share one)
  slot_ref[slot[j]] = (int)vals[j];
  int i0 = idx[3 * (int64_t)t], i1 = idx[3 * (int64_t)t + 1], i2 = idx[3 * (int64_t)t + 2];
  float v0[3], e1[3], e2[3];
  for (int a = 0; a < 3; ++a) {
    v0[a] = xyz[3 * (int64_t)i0 + a];
    e1[a] = xyz[3 * (int64_t)i1 + a] - v0[a];
    e2[a] = xyz[3 * (int64_t)i2 + a] - v0[a];
  }
  float4* o = tris + 3 * (int64_t)slot[j];
  o[0] = make_float4(v0[0], v0[1], v0[2], e1[0]);
  o[1] = make_float4(e1[1], e1[2], e2[0], e2[1]);
  o[2] = make_float4(e2[2], __int_as_float(t), __uint_as_float(code[t]), __int_as_float(chan[t]));
}


// ---- refit (dw_refit_bvh): same triangles, same tree, new vertex positions.
// errs[0] triangles with a non-finite vertex, errs[1] with zero area (the tests of dw_set_geometry), errs[2] first bad triangle
__global__ void refit_check_kernel(int n, const float* __restrict__ xyz, const int32_t* __restrict__ idx,
                                   unsigned long long* __restrict__ errs) {
  int t = blockIdx.x * blockDim.x + threadIdx.x;
  if (t >= n) return;
  float v[3][3];
  load_tri(xyz, idx, t, v);
  bool fin = true;
  for (int k = 0; k < 3; ++k) for (int a = 0; a < 3; ++a) fin = fin && isfinite(v[k][a]);
  if (!fin) { atomicAdd(&errs[0], 1ull); atomicMin(&errs[2], (unsigned long long)t); return; }
  double e1[3], e2[3];
  for (int a = 0; a < 3; ++a) { e1[a] = (double)v[1][a] - v[0][a]; e2[a] = (double)v[2][a] - v[0][a]; }
  double cx = e1[1] * e2[2] - e1[2] * e2[1], cy = e1[2] * e2[0] - e1[0] * e2[2], cz = e1[0] * e2[1] - e1[1] * e2[0];
  if (!(cx * cx + cy * cy + cz * cz > 0.0)) { atomicAdd(&errs[1], 1ull); atomicMin(&errs[2], (unsigned long long)t); }
}
// Boxes of the references of triangle t at its new position.  A split triangle is clipped again; its pieces need not be the
// old ones (any set of boxes whose union covers the triangle is valid: every leaf tests the whole triangle), but the tree has a
// fixed number of references for it: with too many pieces the triangle is split more coarsely, with too few some pieces serve two references.
__global__ void refit_refs_kernel(int n, const float* __restrict__ xyz, const int32_t* __restrict__ idx,
                                  const float* __restrict__ tlo, const float* __restrict__ thi,
                                  const unsigned* __restrict__ scene, int split_div, float pad, const int* __restrict__ offs,
                                  const int* __restrict__ counts, float* __restrict__ rlo, float* __restrict__ rhi,
                                  int* __restrict__ n_loose) {
  int t = blockIdx.x * blockDim.x + threadIdx.x;
  if (t >= n) return;
  const int o = offs[t], cnt = counts[t];
  const float* lo = tlo + 3 * (int64_t)t;
  const float* hi = thi + 3 * (int64_t)t;
  float* olo = rlo + 3 * (int64_t)o;
  float* ohi = rhi + 3 * (int64_t)o;
  if (cnt == 1) {
    for (int c = 0; c < 3; ++c) { olo[c] = lo[c]; ohi[c] = hi[c]; }
    return;
  }
  float v[3][3];
  load_tri(xyz, idx, t, v);
  float smax = split_smax(scene, split_div);
  const int want = split_triangle(v, lo, hi, smax, 0.f, nullptr, nullptr);
  int made = want;
  for (int it = 0; made > cnt && it < 16; ++it) {                // more pieces than references: split more coarsely
    smax *= 1.19f;
    made = split_triangle(v, lo, hi, smax, 0.f, nullptr, nullptr);
  }
  made = split_triangle(v, lo, hi, smax, pad, olo, ohi, cnt);    // cap: a last resort, pieces beyond it are merged
  if (made == 1 && cnt > 1)                                      // no longer split: the one box is unpadded, pad it like the others
    for (int c = 0; c < 3; ++c) { olo[c] -= pad; ohi[c] += pad; }
  // fewer pieces than references: reference k takes piece k * made / cnt.  Every piece is used, and since old and new pieces
  // come in the same order along the triangle, a reference keeps a box near the leaf it sits in.  Back to front, in place.
  if (made < cnt)
    for (int k = cnt - 1; k >= 0; --k) {
      const int j = (int)((int64_t)k * made / cnt);
      for (int c = 0; c < 3; ++c) { olo[3 * k + c] = olo[3 * j + c]; ohi[3 * k + c] = ohi[3 * j + c]; }
    }
  if (want != cnt) atomicAdd(n_loose, 1);
}
// Triangle records at the new positions; the triangle of a slot is the caller id its record carries.
__global__ void refit_pack_kernel(int n, const float* __restrict__ xyz, const int32_t* __restrict__ idx, float4* __restrict__ tris) {
  int s = blockIdx.x * blockDim.x + threadIdx.x;
  if (s >= n) return;
  float4* o = tris + 3 * (int64_t)s;
  const float4 c = o[2];
  const int t = __float_as_int(c.y);
  float v[3][3];
  load_tri(xyz, idx, t, v);
  float e1[3], e2[3];
  for (int a = 0; a < 3; ++a) { e1[a] = v[1][a] - v[0][a]; e2[a] = v[2][a] - v[0][a]; }
  o[0] = make_float4(v[0][0], v[0][1], v[0][2], e1[0]);
  o[1] = make_float4(e1[1], e1[2], e2[0], e2[1]);
  o[2] = make_float4(e2[2], c.y, c.z, c.w);
}
// One level of the wide tree, deepest first: the box of a leaf child is the union of the boxes of its references, the box
// of an internal child the union of that node's child boxes (already recomputed: children have larger indices and lie deeper).
__global__ void refit_level_kernel(int first, int count, float4* __restrict__ nodes, const int* __restrict__ slot_ref,
                                   const float* __restrict__ rlo, const float* __restrict__ rhi) {
  int i = blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= count) return;
  const int w = first + i;
  const float4 rf = nodes[8 * (int64_t)w + 6];
  const int ref[4] = {__float_as_int(rf.x), __float_as_int(rf.y), __float_as_int(rf.z), __float_as_int(rf.w)};
  float4 lo[4], hi[4];
  for (int k = 0; k < 4; ++k) {
    lo[k] = make_float4(FLT_MAX, FLT_MAX, FLT_MAX, 0.f); hi[k] = make_float4(-FLT_MAX, -FLT_MAX, -FLT_MAX, 0.f);
    if (ref[k] == DW_REF_NONE) continue;
    if (ref[k] < 0) {
      const int code = ~ref[k], s0 = code >> 3, cnt = (code & 7) + 1;
      for (int s = s0; s < s0 + cnt; ++s) {
        const int64_t r = slot_ref[s];
        lo[k] = min4(lo[k], make_float4(rlo[3 * r], rlo[3 * r + 1], rlo[3 * r + 2], 0.f));
        hi[k] = max4(hi[k], make_float4(rhi[3 * r], rhi[3 * r + 1], rhi[3 * r + 2], 0.f));
      }
    } else {
      const float4* ch = nodes + 8 * (int64_t)ref[k];
      const float4 cr = ch[6];
      const int cref[4] = {__float_as_int(cr.x), __float_as_int(cr.y), __float_as_int(cr.z), __float_as_int(cr.w)};
      const float4 q0 = ch[0], q1 = ch[1], q2 = ch[2], q3 = ch[3], q4 = ch[4], q5 = ch[5];
      const float cl[4][3] = {{q0.x, q1.x, q2.x}, {q0.y, q1.y, q2.y}, {q0.z, q1.z, q2.z}, {q0.w, q1.w, q2.w}};
      const float chh[4][3] = {{q3.x, q4.x, q5.x}, {q3.y, q4.y, q5.y}, {q3.z, q4.z, q5.z}, {q3.w, q4.w, q5.w}};
      for (int j = 0; j < 4; ++j) {
        if (cref[j] == DW_REF_NONE) continue;
        lo[k] = min4(lo[k], make_float4(cl[j][0], cl[j][1], cl[j][2], 0.f));
        hi[k] = max4(hi[k], make_float4(chh[j][0], chh[j][1], chh[j][2], 0.f));
      }
    }
  }
  write_wide(nodes, w, lo, hi, ref);
}

// The 64-byte form of the nodes that the queries read (dw_internal.cuh DwBvh::qnodes): every plane as a 16-bit step of q_cs from
// q_lo, lower planes rounded down and upper planes up, one more step outwards for the rounding of the division.  At 65535 steps
// over the scene a step is 0.04 mm for a 2.6 m detector: the boxes grow by less than the triangles' own padding, and a box only
// decides HOW the nearest hit is found.  Half the bytes per visit: the L1 data pipe (one wavefront per lane and 128 bytes of a
// divergent load) is what bounds the traversal (profiles/r02_experiments.md).
__global__ void quantise_nodes_kernel(int n_nodes, const float4* __restrict__ nodes, uint4* __restrict__ q, float3 qlo, float3 qics) {
  int w = blockIdx.x * blockDim.x + threadIdx.x;
  if (w >= n_nodes) return;
  const float4* p = nodes + 8 * (int64_t)w;
  const float org[3] = {qlo.x, qlo.y, qlo.z}, ics[3] = {qics.x, qics.y, qics.z};
  const float4 rf = p[6];
  const int ref[4] = {__float_as_int(rf.x), __float_as_int(rf.y), __float_as_int(rf.z), __float_as_int(rf.w)};
  unsigned pl[6][4];
  for (int a = 0; a < 3; ++a) {
    const float4 lo = p[a], hi = p[3 + a];
    const float l4[4] = {lo.x, lo.y, lo.z, lo.w}, h4[4] = {hi.x, hi.y, hi.z, hi.w};
    for (int c = 0; c < 4; ++c) {
      if (ref[c] == DW_REF_NONE) { pl[a][c] = 65535u; pl[3 + a][c] = 0u; continue; }
      const float fl = floorf((l4[c] - org[a]) * ics[a]) - 1.0f, fh = ceilf((h4[c] - org[a]) * ics[a]) + 1.0f;
      pl[a][c] = (unsigned)fminf(fmaxf(fl, 0.f), 65535.f);
      pl[3 + a][c] = (unsigned)fminf(fmaxf(fh, 0.f), 65535.f);
    }
  }
  auto pack = [&](int k, int c) { return pl[k][c] | (pl[k][c + 1] << 16); };
  uint4* o = q + 4 * (int64_t)w;
  o[0] = make_uint4(pack(0, 0), pack(0, 2), pack(1, 0), pack(1, 2));
  o[1] = make_uint4(pack(2, 0), pack(2, 2), pack(3, 0), pack(3, 2));
  o[2] = make_uint4(pack(4, 0), pack(4, 2), pack(5, 0), pack(5, 2));
  o[3] = make_uint4((unsigned)ref[0], (unsigned)ref[1], (unsigned)ref[2], (unsigned)ref[3]);
}

// Sum over all nodes of the half-areas of their child boxes: the surface-area measure of tree quality (the expected number of box
// tests of a random ray is proportional to it).  dw_refit_bvh reports it relative to the build.
__global__ void node_area_kernel(int n_nodes, const float4* __restrict__ nodes, double* __restrict__ sum) {
  int w = blockIdx.x * blockDim.x + threadIdx.x;
  double a = 0.0;
  if (w < n_nodes) {
    const float4* p = nodes + 8 * (int64_t)w;
    const float4 q0 = p[0], q1 = p[1], q2 = p[2], q3 = p[3], q4 = p[4], q5 = p[5], rf = p[6];
    if (__float_as_int(rf.x) != DW_REF_NONE) a += half_area(make_float4(q0.x, q1.x, q2.x, 0.f), make_float4(q3.x, q4.x, q5.x, 0.f));
    if (__float_as_int(rf.y) != DW_REF_NONE) a += half_area(make_float4(q0.y, q1.y, q2.y, 0.f), make_float4(q3.y, q4.y, q5.y, 0.f));
    if (__float_as_int(rf.z) != DW_REF_NONE) a += half_area(make_float4(q0.z, q1.z, q2.z, 0.f), make_float4(q3.z, q4.z, q5.z, 0.f));
    if (__float_as_int(rf.w) != DW_REF_NONE) a += half_area(make_float4(q0.w, q1.w, q2.w, 0.f), make_float4(q3.w, q4.w, q5.w, 0.f));
  }
  for (int o = 16; o; o >>= 1) a += __shfl_xor_sync(0xffffffffu, a, o);
  if ((threadIdx.x & 31) == 0 && a != 0.0) atomicAdd(sum, a);
}

// ---- empty-space grid.  G^3 cells over the scene box.  A cell is OCCUPIED if the box of any
// triangle, grown by `margin`, overlaps it.  Every free cell gets one axis-aligned box of free cells that contains it
// (grown greedily, one layer of cells at a time, faces in turn); a ray segment whose two ends lie in that box cannot touch
// a triangle, so the propagation kernel answers such a query without traversal.  Conservative by construction: margin is
// larger than every tolerance the traversal uses (edge slack, eps_len, fp32 rounding of the end point).
__global__ void grid_mark_kernel(int n, const float* __restrict__ tlo, const float* __restrict__ thi, float3 glo, float3 inv_cs,
                                 float margin, int G, int* __restrict__ occ) {
  int t = blockIdx.x * blockDim.x + threadIdx.x;
  if (t >= n) return;
  int c0[3], c1[3];
  const float g[3] = {glo.x, glo.y, glo.z}, ic[3] = {inv_cs.x, inv_cs.y, inv_cs.z};
  for (int a = 0; a < 3; ++a) {
    float lo = (tlo[3 * (int64_t)t + a] - margin - g[a]) * ic[a], hi = (thi[3 * (int64_t)t + a] + margin - g[a]) * ic[a];
    c0[a] = min(max((int)floorf(lo), 0), G - 1);
    c1[a] = min(max((int)floorf(hi), 0), G - 1);
  }
  for (int k = c0[2]; k <= c1[2]; ++k)
    for (int j = c0[1]; j <= c1[1]; ++j)
      for (int i = c0[0]; i <= c1[0]; ++i) occ[(k * G + j) * G + i] = 1;
}

// Summed-area table S[(k+1),(j+1),(i+1)] = number of occupied cells in [0..i] x [0..j] x [0..k]; borders are zero.
__global__ void sat_x_kernel(int G, const int* __restrict__ occ, int* __restrict__ S) {
  int id = blockIdx.x * blockDim.x + threadIdx.x;
  if (id >= G * G) return;
  int j = id % G, k = id / G, P = G + 1, run = 0;
  for (int i = 0; i < G; ++i) { run += occ[(k * G + j) * G + i]; S[((k + 1) * P + (j + 1)) * P + (i + 1)] = run; }
}
__global__ void sat_y_kernel(int G, int* __restrict__ S) {
  int id = blockIdx.x * blockDim.x + threadIdx.x;
  if (id >= G * G) return;
  int i = id % G, k = id / G, P = G + 1, run = 0;
  for (int j = 0; j < G; ++j) { int* p = &S[((k + 1) * P + (j + 1)) * P + (i + 1)]; run += *p; *p = run; }
}
__global__ void sat_z_kernel(int G, int* __restrict__ S) {
  int id = blockIdx.x * blockDim.x + threadIdx.x;
  if (id >= G * G) return;
  int i = id % G, j = id / G, P = G + 1, run = 0;
  for (int k = 0; k < G; ++k) { int* p = &S[((k + 1) * P + (j + 1)) * P + (i + 1)]; run += *p; *p = run; }
}
__device__ __forceinline__ int sat_sum(const int* __restrict__ S, int P, int x0, int x1, int y0, int y1, int z0, int z1) {
  auto at = [&](int k, int j, int i) { return S[(k * P + j) * P + i]; };
  return at(z1 + 1, y1 + 1, x1 + 1) - at(z0, y1 + 1, x1 + 1) - at(z1 + 1, y0, x1 + 1) - at(z1 + 1, y1 + 1, x0) +
         at(z0, y0, x1 + 1) + at(z0, y1 + 1, x0) + at(z1 + 1, y0, x0) - at(z0, y0, x0);
}
// cells[c] = (x0 | x1<<8 | y0<<16 | y1<<24, z0 | z1<<8 | valid<<16): inclusive cell bounds of the free box of cell c.
__global__ void grid_grow_kernel(int G, const int* __restrict__ occ, const int* __restrict__ S, uint2* __restrict__ cells,
                                 int* __restrict__ n_free) {
  int c = blockIdx.x * blockDim.x + threadIdx.x;
  if (c >= G * G * G) return;
  if (occ[c]) { cells[c] = make_uint2(0u, 0u); return; }
  const int P = G + 1;
  int b[6] = {c % G, c % G, (c / G) % G, (c / G) % G, c / (G * G), c / (G * G)};   // x0 x1 y0 y1 z0 z1
  bool grew = true;
  while (grew) {
    grew = false;
    for (int f = 0; f < 6; ++f) {
      const bool low = (f & 1) == 0;
      if (low ? b[f] == 0 : b[f] == G - 1) continue;
      int s[6] = {b[0], b[1], b[2], b[3], b[4], b[5]};
      const int layer = low ? b[f] - 1 : b[f] + 1;
      s[f & ~1] = layer; s[f | 1] = layer;                                         // the one-cell layer next to face f
      if (sat_sum(S, P, s[0], s[1], s[2], s[3], s[4], s[5]) == 0) { b[f] = layer; grew = true; }
    }
  }
  cells[c] = make_uint2((unsigned)b[0] | (unsigned)b[1] << 8 | (unsigned)b[2] << 16 | (unsigned)b[3] << 24,
                        (unsigned)b[4] | (unsigned)b[5] << 8 | 1u << 16);
  atomicAdd(n_free, 1);
}

}  // namespace

// Stream-ordered allocation from the context's pool, which keeps its memory: a build makes about forty buffers, and cudaMalloc /
// cudaFree (each a device synchronisation) were most of its time.  What a build leaves behind is freed with cudaFree (dw_bvh_free).
template <class T> static cudaError_t dw_salloc(dw_ctx* c, T** p, size_t bytes, cudaStream_t s) {
  if (bytes == 0) bytes = 4;
  return c->pool ? cudaMallocFromPoolAsync((void**)p, bytes, c->pool, s) : cudaMallocAsync((void**)p, bytes, s);
}
static void dw_sfree(void* p, cudaStream_t s) { if (p) cudaFreeAsync(p, s); }

static inline unsigned G_blocks(int64_t n, int B) { return (unsigned)((n + B - 1) / B); }

#define DW_B(call) do { cudaError_t e__ = (call); if (e__ != cudaSuccess) { rc = dw_fail(c, DW_E_CUDA, "%s failed: %s (%s:%d)", \
    #call, cudaGetErrorString(e__), __FILE__, __LINE__); goto done; } } while (0)


// Empty-space grid over the scene box [lo, hi] from the reference boxes (rebuilt as a whole by a refit); nothing is built for an
// empty or flat world.  c->d_cells is allocated here if it is not there yet (GR^3 cells; a refit keeps the resolution).
static int grid_build(dw_ctx* c, int n, const float* tlo, const float* thi, const float lo[3], const float hi[3], float eps_len,
                      int GR, cudaStream_t stream, int* grid_built, int* grid_free, float* grid_ms) {
  int rc = DW_OK;
  const int B = 256;
  int *occ = nullptr, *sat = nullptr, *cnt = nullptr;
  cudaEvent_t ev0 = nullptr, ev1 = nullptr;
  *grid_built = 0; *grid_free = 0; *grid_ms = 0.f;
  c->bvh.cells = nullptr; c->bvh.grid_n = 0;
  float ext[3] = {hi[0] - lo[0], hi[1] - lo[1], hi[2] - lo[2]};
  const float emax = fmaxf(ext[0], fmaxf(ext[1], ext[2]));
  if (n <= 0 || !(emax > 0.f)) return DW_OK;
  {
    for (int a = 0; a < 3; ++a) ext[a] = fmaxf(ext[a], 1e-3f * emax);           // a flat axis still gets cells of finite size
    const float3 glo = make_float3(lo[0], lo[1], lo[2]);
    const float3 cs = make_float3(ext[0] / GR, ext[1] / GR, ext[2] / GR);
    const float3 ics = make_float3(GR / ext[0], GR / ext[1], GR / ext[2]);
    // margin > edge slack (2e-6 x longest edge <= 15 eps_len) + eps_len of t_max + fp32 rounding of the segment end
    const float margin = 32.0f * eps_len;
    const int G3 = GR * GR * GR, P = GR + 1;
    DW_B(cudaEventCreate(&ev0)); DW_B(cudaEventCreate(&ev1));
    DW_B(dw_salloc(c, &occ, 4 * (size_t)G3, stream)); DW_B(dw_salloc(c, &sat, 4 * (size_t)P * P * P, stream)); DW_B(dw_salloc(c, &cnt, 4, stream));
    if (!c->d_cells) DW_B(dw_salloc(c, &c->d_cells, sizeof(uint2) * (size_t)G3, stream));
    DW_B(cudaMemsetAsync(occ, 0, 4 * (size_t)G3, stream));
    DW_B(cudaMemsetAsync(sat, 0, 4 * (size_t)P * P * P, stream));
    DW_B(cudaMemsetAsync(cnt, 0, 4, stream));
    DW_B(cudaEventRecord(ev0, stream));
    grid_mark_kernel<<<G_blocks(n, B), B, 0, stream>>>(n, tlo, thi, glo, ics, margin, GR, occ);
    sat_x_kernel<<<G_blocks(GR * GR, B), B, 0, stream>>>(GR, occ, sat);
    sat_y_kernel<<<G_blocks(GR * GR, B), B, 0, stream>>>(GR, sat);
    sat_z_kernel<<<G_blocks(GR * GR, B), B, 0, stream>>>(GR, sat);
    grid_grow_kernel<<<G_blocks(G3, B), B, 0, stream>>>(GR, occ, sat, c->d_cells, cnt);
    DW_B(cudaGetLastError());
    DW_B(cudaEventRecord(ev1, stream));
    DW_B(cudaMemcpyAsync(grid_free, cnt, 4, cudaMemcpyDeviceToHost, stream));
    DW_B(cudaStreamSynchronize(stream));
    cudaEventElapsedTime(grid_ms, ev0, ev1);
    *grid_built = GR;
    c->bvh.cells = c->d_cells; c->bvh.grid_n = GR; c->bvh.grid_lo = glo; c->bvh.grid_cs = cs; c->bvh.grid_inv_cs = ics;
  }
done:
  dw_sfree(occ, stream); dw_sfree(sat, stream); dw_sfree(cnt, stream);
  if (ev0) cudaEventDestroy(ev0);
  if (ev1) cudaEventDestroy(ev1);
  return rc;
}

// (re)writes c->d_qnodes from c->d_nodes for the scene box [lo, hi]
static int quantise_nodes(dw_ctx* c, int n_nodes, const float lo[3], const float hi[3], cudaStream_t stream) {
  if (!DW_NODE_Q16) return DW_OK;
  if (!c->d_qnodes) DW_CUDA(c, dw_salloc(c, &c->d_qnodes, 64 * (size_t)std::max(n_nodes, 1), stream));
  float3 qlo, qcs, qics;
  float* l = &qlo.x; float* s = &qcs.x; float* is = &qics.x;
  for (int a = 0; a < 3; ++a) {
    const float ext = hi[a] - lo[a], pad = 1e-3f * ext + 1e-3f;      // node boxes carry the padding of the references
    l[a] = lo[a] - pad;
    s[a] = (ext + 2.0f * pad) / 65535.0f;
    is[a] = 1.0f / s[a];
  }
  quantise_nodes_kernel<<<G_blocks(n_nodes, 256), 256, 0, stream>>>(n_nodes, c->d_nodes, c->d_qnodes, qlo, qics);
  DW_CUDA(c, cudaGetLastError());
  c->bvh.qnodes = c->d_qnodes; c->bvh.q_lo = qlo; c->bvh.q_cs = qcs;
  return DW_OK;
}

#if DW_WIDE8
// Experiment: the 4-wide tree re-made 8-wide on the host (dw_internal.cuh DW_WIDE8).  Replaces c->d_nodes; the refit state is void.
static int widen8(dw_ctx* c, int n_nodes, cudaStream_t stream, int* n8_out) {
  struct Child { float lo[3], hi[3]; int ref; };
  std::vector<float4> h(8 * (size_t)n_nodes);
  DW_CUDA(c, cudaStreamSynchronize(stream));
  DW_CUDA(c, cudaMemcpy(h.data(), c->d_nodes, sizeof(float4) * h.size(), cudaMemcpyDeviceToHost));
  auto kids = [&](int node, std::vector<Child>& out) {
    const float* q = reinterpret_cast<const float*>(&h[8 * (size_t)node]);
    for (int k = 0; k < 4; ++k) {
      int ref; memcpy(&ref, q + 24 + k, 4);
      if (ref == DW_REF_NONE) continue;
      Child ch;
      for (int a = 0; a < 3; ++a) { ch.lo[a] = q[4 * a + k]; ch.hi[a] = q[12 + 4 * a + k]; }
      ch.ref = ref;
      out.push_back(ch);
    }
  };
  auto count4 = [&](int node) { std::vector<Child> t; kids(node, t); return (int)t.size(); };
  auto area = [](const Child& ch) { const float x = ch.hi[0] - ch.lo[0], y = ch.hi[1] - ch.lo[1], z = ch.hi[2] - ch.lo[2]; return x * y + y * z + z * x; };
  std::vector<int> from{0};                       // 8-wide node -> the 4-wide node it starts from
  std::vector<float4> out;
  for (size_t i = 0; i < from.size(); ++i) {
    std::vector<Child> L;
    kids(from[i], L);
    for (;;) {                                    // pull up the children of the largest inner child that still fits
      int best = -1;
      for (int k = 0; k < (int)L.size(); ++k)
        if (L[k].ref >= 0 && (int)L.size() - 1 + count4(L[k].ref) <= 8 && (best < 0 || area(L[k]) > area(L[best]))) best = k;
      if (best < 0) break;
      const int node = L[best].ref;
      L.erase(L.begin() + best);
      kids(node, L);
    }
    for (Child& ch : L)
      if (ch.ref >= 0) { from.push_back(ch.ref); ch.ref = (int)from.size() - 1; }
    float rec[64];
    for (int half = 0; half < 2; ++half)
      for (int k = 0; k < 4; ++k) {
        const int j = 4 * half + k;
        const bool on = j < (int)L.size();
        float* q = rec + 32 * half;
        for (int a = 0; a < 3; ++a) { q[4 * a + k] = on ? L[j].lo[a] : FLT_MAX; q[12 + 4 * a + k] = on ? L[j].hi[a] : -FLT_MAX; }
        const int ref = on ? L[j].ref : DW_REF_NONE;
        memcpy(q + 24 + k, &ref, 4);
        q[28 + k] = 0.f;
      }
    for (int v = 0; v < 16; ++v) out.push_back(make_float4(rec[4 * v], rec[4 * v + 1], rec[4 * v + 2], rec[4 * v + 3]));
  }
  float4* d = nullptr;
  DW_CUDA(c, cudaMalloc(&d, sizeof(float4) * out.size()));
  DW_CUDA(c, cudaMemcpy(d, out.data(), sizeof(float4) * out.size(), cudaMemcpyHostToDevice));
  cudaFree(c->d_nodes);
  c->d_nodes = d;
  *n8_out = (int)from.size();
  return DW_OK;
}
#endif

static int nodes_area(dw_ctx* c, int n_nodes, cudaStream_t stream, double* out) {
  int rc = DW_OK;
  double* d = nullptr;
  *out = 0.0;
  DW_B(dw_salloc(c, &d, 8, stream));
  DW_B(cudaMemsetAsync(d, 0, 8, stream));
  node_area_kernel<<<G_blocks(n_nodes, 256), 256, 0, stream>>>(n_nodes, c->d_nodes, d);
  DW_B(cudaGetLastError());
  DW_B(cudaMemcpyAsync(out, d, 8, cudaMemcpyDeviceToHost, stream));
  DW_B(cudaStreamSynchronize(stream));
done:
  dw_sfree(d, stream);
  return rc;
}

void dw_bvh_free(dw_ctx* c) {
  cudaFree(c->d_nodes); cudaFree(c->d_qnodes); cudaFree(c->d_tris); cudaFree(c->d_cells);
  c->d_nodes = nullptr; c->d_qnodes = nullptr; c->d_tris = nullptr; c->d_cells = nullptr; c->built = false;
  dw_ctx::Refit& r = c->rf;
  cudaFree(r.counts); cudaFree(r.offs); cudaFree(r.slot_ref); cudaFree(r.tlo); cudaFree(r.thi); cudaFree(r.rlo); cudaFree(r.rhi);
  cudaFree(r.scene);
  r = dw_ctx::Refit{};
}

int dw_bvh_build_impl(dw_ctx* c, const dw_build_params* params, dw_build_stats* stats, cudaStream_t stream) {
  int rc = DW_OK;
  const int nt = (int)c->n_tri;     // triangles
  int n = nt;                       // references (>= nt once long triangles are split): what the tree is built over
  const int max_leaf = (params && params->max_leaf_tris) ? params->max_leaf_tris : 2;
  const int radius = (params && params->ploc_radius) ? params->ploc_radius : 16;
  if (max_leaf < 1 || max_leaf > 8) return dw_fail(c, DW_E_ARG, "dw_build_bvh: max_leaf_tris must be in 1..8");
  if (radius < 1 || radius > 256) return dw_fail(c, DW_E_ARG, "dw_build_bvh: ploc_radius must be in 1..256");
  const int grid_req = params ? params->grid_res : 0;
  const int GR = grid_req == 0 ? 64 : grid_req;
  const int split_req = params ? params->split_div : 0;
  const int split_div = split_req == 0 ? 32 : split_req;
  if (split_req != -1 && (split_div < 1 || split_div > 4096)) return dw_fail(c, DW_E_ARG, "dw_build_bvh: split_div must be -1, 0 or in 1..4096");
  if (grid_req != -1 && (GR < 8 || GR > 128)) return dw_fail(c, DW_E_ARG, "dw_build_bvh: grid_res must be -1, 0 or in 8..128");
  dw_bvh_free(c);
  if (stats) memset(stats, 0, sizeof *stats);

  size_t N = 0, N2 = 0;             // set after stage 0
  const size_t NT = (size_t)std::max(nt, 1);
  float *tlo = nullptr, *thi = nullptr, *tlo_t = nullptr, *thi_t = nullptr;   // tlo/thi: boxes of the references; *_t: of the triangles
  int *counts = nullptr, *offs = nullptr, *ref_tri = nullptr;
  float4 *blo = nullptr, *bhi = nullptr, *cl[2] = {nullptr, nullptr}, *ch[2] = {nullptr, nullptr}, *nodes_tmp = nullptr;
  unsigned *scene = nullptr, *vals = nullptr, *vals2 = nullptr;
  unsigned long long *keys = nullptr, *keys2 = nullptr;
  int *left = nullptr, *right = nullptr, *parent = nullptr, *size = nullptr, *leftmost = nullptr, *cn[2] = {nullptr, nullptr},
      *nn = nullptr, *slot = nullptr, *misc = nullptr, *occ = nullptr, *sat = nullptr, *pst = nullptr;
  unsigned char* flag = nullptr;
  int2 *bsum = nullptr, *boff = nullptr;
  constexpr int kMaxWideLevels = 48;   // more levels than the traversal stack allows: the depth check below refuses such a tree
  int grid_built = 0, grid_free = 0, split_used = 0;
  WideTask* tasks[2] = {nullptr, nullptr};
  void* tmp = nullptr;
  size_t tmp_bytes = 0, tmp2 = 0;
  cudaEvent_t ev0 = nullptr, ev1 = nullptr;
  unsigned h_scene[6] = {0, 0, 0, 0, 0, 0};
  int h_misc[4] = {0, 0, 0, 0};      // [0] next-level tasks, [1] wide nodes, [2] leaves, [3] binary depth
  int n_nodes = 1, wide_depth = 1, ploc_rounds = 0;
  std::vector<int> levels{0, 1};     // wide-tree level k = nodes [levels[k], levels[k+1]) (kept for dw_refit_bvh)
  const int B = 256;
  unsigned G = 0;
  const unsigned GT = (unsigned)((NT + B - 1) / B);

  DW_B(cudaEventCreate(&ev0)); DW_B(cudaEventCreate(&ev1));
  DW_B(dw_salloc(c, &scene, sizeof(unsigned) * 6, stream));
  DW_B(dw_salloc(c, &misc, 16, stream));
  DW_B(cudaEventRecord(ev0, stream));
  DW_B(cudaMemsetAsync(misc, 0, 16, stream));
  // ---- stage 0: triangle boxes, scene bounds, references (long triangles split)
  DW_B(dw_salloc(c, &tlo_t, sizeof(float) * 3 * NT, stream)); DW_B(dw_salloc(c, &thi_t, sizeof(float) * 3 * NT, stream));
  DW_B(dw_salloc(c, &counts, 4 * NT, stream)); DW_B(dw_salloc(c, &offs, 4 * NT, stream));
  if (nt > 0) {
    unsigned init[6] = {0xffffffffu, 0xffffffffu, 0xffffffffu, 0u, 0u, 0u};
    DW_B(cudaMemcpyAsync(scene, init, sizeof init, cudaMemcpyHostToDevice, stream));
    tri_bounds_kernel<<<GT, B, 0, stream>>>(nt, c->d_xyz, c->d_idx, tlo_t, thi_t, scene);
    DW_B(cudaMemcpyAsync(h_scene, scene, sizeof h_scene, cudaMemcpyDeviceToHost, stream));
    DW_B(cudaStreamSynchronize(stream));
    float mx0 = 0.f;
    for (int a = 0; a < 6; ++a) mx0 = fmaxf(mx0, fabsf(o2f(h_scene[a])));
    const float pad = 4.0f * 1.1920929e-7f * mx0;               // = eps_len: boxes of split references are padded by it
    int div = split_req == -1 ? 0 : split_div;
    size_t scan_bytes = 0;
    DW_B(cub::DeviceScan::ExclusiveSum(nullptr, scan_bytes, counts, offs, nt, stream));
    DW_B(dw_salloc(c, &tmp, scan_bytes, stream));
    for (;;) {                                                  // coarser splitting if the references would more than double
      split_count_kernel<<<GT, B, 0, stream>>>(nt, c->d_xyz, c->d_idx, tlo_t, thi_t, scene, div, counts);
      DW_B(cub::DeviceScan::ExclusiveSum(tmp, scan_bytes, counts, offs, nt, stream));
      int h_last[2];
      DW_B(cudaMemcpyAsync(&h_last[0], offs + (nt - 1), 4, cudaMemcpyDeviceToHost, stream));
      DW_B(cudaMemcpyAsync(&h_last[1], counts + (nt - 1), 4, cudaMemcpyDeviceToHost, stream));
      DW_B(cudaStreamSynchronize(stream));
      n = h_last[0] + h_last[1];
      if (div <= 1 || (int64_t)n <= 2 * (int64_t)nt + 65536) break;
      div /= 2;
    }
    split_used = div;
    if (n < 0 || n >= (1 << 28)) {                              // a leaf reference is (slot << 3) | (count - 1) in 31 bits
      rc = dw_fail(c, DW_E_RANGE, "dw_build_bvh: %d box references (limit 2^28)", n);
      goto done;
    }
    DW_B(dw_salloc(c, &tlo, sizeof(float) * 3 * (size_t)n, stream)); DW_B(dw_salloc(c, &thi, sizeof(float) * 3 * (size_t)n, stream));
    DW_B(dw_salloc(c, &ref_tri, 4 * (size_t)n, stream));
    split_emit_kernel<<<GT, B, 0, stream>>>(nt, c->d_xyz, c->d_idx, tlo_t, thi_t, scene, div, pad, offs, counts, tlo, thi, ref_tri);
    dw_sfree(tmp, stream); tmp = nullptr;
  }
  N = (size_t)std::max(n, 1); N2 = 2 * N;
  G = (unsigned)((N + B - 1) / B);
  {   // grow the pool once for everything that follows (about 390 bytes per reference): forty small growths cost a first build 5 ms
    void* warm = nullptr;
    if (dw_salloc(c, &warm, 400 * N + (1 << 20), stream) == cudaSuccess) dw_sfree(warm, stream); else cudaGetLastError();
  }
  DW_B(dw_salloc(c, &blo, sizeof(float4) * N2, stream)); DW_B(dw_salloc(c, &bhi, sizeof(float4) * N2, stream));
  for (int k = 0; k < 2; ++k) {
    DW_B(dw_salloc(c, &cl[k], sizeof(float4) * N, stream)); DW_B(dw_salloc(c, &ch[k], sizeof(float4) * N, stream)); DW_B(dw_salloc(c, &cn[k], 4 * N, stream));
    DW_B(dw_salloc(c, &tasks[k], sizeof(WideTask) * N, stream));
  }
  DW_B(dw_salloc(c, &keys, 8 * N, stream)); DW_B(dw_salloc(c, &keys2, 8 * N, stream));
  DW_B(dw_salloc(c, &vals, 4 * N, stream)); DW_B(dw_salloc(c, &vals2, 4 * N, stream));
  DW_B(dw_salloc(c, &left, 4 * N2, stream)); DW_B(dw_salloc(c, &right, 4 * N2, stream)); DW_B(dw_salloc(c, &parent, 4 * N2, stream));
  DW_B(dw_salloc(c, &size, 4 * N2, stream)); DW_B(dw_salloc(c, &leftmost, 4 * N2, stream));
  DW_B(dw_salloc(c, &nn, 4 * N, stream)); DW_B(dw_salloc(c, &flag, N, stream)); DW_B(dw_salloc(c, &slot, 4 * N, stream));
  DW_B(dw_salloc(c, &bsum, sizeof(int2) * (N / 256 + 1), stream)); DW_B(dw_salloc(c, &boff, sizeof(int2) * (N / 256 + 1), stream));
  DW_B(dw_salloc(c, &pst, 4 * (8 + kMaxWideLevels + 2), stream));
  DW_B(cub::DeviceRadixSort::SortPairs(nullptr, tmp_bytes, keys, keys2, vals, vals2, (int)N, 0, 63, stream));
  (void)tmp2;
  DW_B(dw_salloc(c, &tmp, tmp_bytes, stream));
  DW_B(dw_salloc(c, &c->d_tris, 48 * N, stream));
  DW_B(dw_salloc(c, &c->rf.slot_ref, 4 * N, stream));

  if (n > 0) {
    morton_kernel<<<G, B, 0, stream>>>(n, tlo, thi, scene, keys, vals);
    DW_B(cub::DeviceRadixSort::SortPairs(tmp, tmp_bytes, keys, keys2, vals, vals2, n, 0, 63, stream));
    ploc_init_kernel<<<G, B, 0, stream>>>(n, vals2, tlo, thi, blo, bhi, cn[0], cl[0], ch[0], size, parent, leftmost);
    // ---- PLOC rounds: clusters [0, m) in buffer `cur`; every round makes at least one node.  m and the next node index are on the
    // device (pst[0..1] / pst[2..3] by the parity of the round, pst[4] rounds, pst[5] error); one read-back per chunk of rounds
    int base = n;
    {
      int init[8] = {n, n, n, n, 0, 0, 0, 0};
      DW_B(cudaMemcpyAsync(pst, init, sizeof init, cudaMemcpyHostToDevice, stream));
      int m = n, r = 0;
      while (m > 1) {
        if (r > 8192) { rc = dw_fail(c, DW_E_CUDA, "dw_build_bvh: clustering does not end"); goto done; }
        const int chunk = r == 0 ? 24 : 12;
        for (int q = 0; q < chunk; ++q, ++r) {
          const int* st = pst + 2 * (r & 1);
          int* stn = pst + 2 * ((r + 1) & 1);
          const int cur = r & 1;
          ploc_nn_kernel_dev<<<G, B, 0, stream>>>(st, radius, cl[cur], ch[cur], nn);
          ploc_mark_kernel_dev<<<G, B, 0, stream>>>(st, nn, flag, bsum);
          ploc_scan_kernel_dev<<<1, 1024, 0, stream>>>(st, stn, pst + 4, bsum, boff);
          ploc_apply_kernel_dev<<<G, B, 0, stream>>>(st, nn, flag, boff, cn[cur], cl[cur], ch[cur], cn[cur ^ 1], cl[cur ^ 1], ch[cur ^ 1],
                                                     left, right, parent, blo, bhi, size);
        }
        int h[8];
        DW_B(cudaMemcpyAsync(h, pst, sizeof h, cudaMemcpyDeviceToHost, stream));
        DW_B(cudaStreamSynchronize(stream));
        if (h[5]) { rc = dw_fail(c, DW_E_CUDA, "dw_build_bvh: a clustering round made no progress"); goto done; }
        m = h[2 * (r & 1)]; base = h[2 * (r & 1) + 1];
        ploc_rounds = h[4] > 0 ? h[4] : ploc_rounds;
      }
      // rounds launched after m reached 1 did nothing, but were counted: the rounds that merged are those until base was complete
    }
    if (base != 2 * n - 1) { rc = dw_fail(c, DW_E_CUDA, "dw_build_bvh: %d of %d nodes made", base - n, n - 1); goto done; }
    leaf_walk_kernel<<<G, B, 0, stream>>>(n, left, parent, size, slot, leftmost, misc + 3);
    pack_tris_kernel<<<G, B, 0, stream>>>(n, vals2, ref_tri, slot, c->d_xyz, c->d_idx, c->d_code, c->d_chan, c->d_tris, c->rf.slot_ref);
  }
  if (n <= max_leaf) {
    DW_B(dw_salloc(c, &c->d_nodes, 128, stream));
    wide_single_kernel<<<1, 1, 0, stream>>>(n, blo, bhi, c->d_nodes);
    h_misc[1] = 1; h_misc[2] = n > 0 ? 1 : 0;
  } else {
    // ---- collapse, one launch per level of the wide tree
    DW_B(dw_salloc(c, &nodes_tmp, 128 * N, stream));
    WideTask t0{2 * n - 2, 0};
    int init[3] = {0, 1, 0};
    int* lvl = pst + 8;                                           // lvl[k] = tasks (= nodes) of level k, counted by the level before
    std::vector<int> h_lvl(kMaxWideLevels + 2, 0);
    h_lvl[0] = 1;
    DW_B(cudaMemcpyAsync(tasks[0], &t0, sizeof t0, cudaMemcpyHostToDevice, stream));
    DW_B(cudaMemcpyAsync(misc, init, sizeof init, cudaMemcpyHostToDevice, stream));
    DW_B(cudaMemcpyAsync(lvl, h_lvl.data(), 4 * (kMaxWideLevels + 2), cudaMemcpyHostToDevice, stream));
    {
      const unsigned Gc = (unsigned)std::min<size_t>((N + B - 1) / B, (size_t)c->sm_count * 8);
      for (int k = 0; k <= kMaxWideLevels; ++k)                   // a level without tasks is an empty launch
        wide_collapse_kernel<<<Gc, B, 0, stream>>>(lvl + k, lvl + k + 1, tasks[k & 1], tasks[(k + 1) & 1], misc, max_leaf, left, right, size, blo, bhi,
                                                   slot, leftmost, nodes_tmp);
      DW_B(cudaMemcpyAsync(h_lvl.data(), lvl, 4 * (kMaxWideLevels + 2), cudaMemcpyDeviceToHost, stream));
      DW_B(cudaStreamSynchronize(stream));
      wide_depth = 0;
      for (int k = 0; k <= kMaxWideLevels + 1 && h_lvl[k] > 0; ++k) {
        ++wide_depth;
        if (k > 0) levels.push_back(levels.back() + h_lvl[k]);  // the children made by level k - 1 are level k
      }
      if (h_lvl[kMaxWideLevels + 1] > 0) { rc = dw_fail(c, DW_E_RANGE, "dw_build_bvh: the tree is deeper than %d levels", kMaxWideLevels); goto done; }
    }
    DW_B(cudaMemcpyAsync(h_misc, misc, 16, cudaMemcpyDeviceToHost, stream));
    DW_B(cudaStreamSynchronize(stream));
    n_nodes = h_misc[1];
    DW_B(dw_salloc(c, &c->d_nodes, 128 * (size_t)n_nodes, stream));
    DW_B(cudaMemcpyAsync(c->d_nodes, nodes_tmp, 128 * (size_t)n_nodes, cudaMemcpyDeviceToDevice, stream));
  }
  DW_B(cudaGetLastError());
  DW_B(cudaEventRecord(ev1, stream));
  if (n > 0) DW_B(cudaMemcpyAsync(h_scene, scene, sizeof h_scene, cudaMemcpyDeviceToHost, stream));
  DW_B(cudaMemcpyAsync(&h_misc[3], misc + 3, 4, cudaMemcpyDeviceToHost, stream));
  DW_B(cudaStreamSynchronize(stream));
  if (3 * wide_depth > kDwStackShared + kDwStackLocal) {
    rc = dw_fail(c, DW_E_RANGE, "dw_build_bvh: tree depth %d exceeds the traversal stack (%d entries)", wide_depth, kDwStackShared + kDwStackLocal);
    goto done;
  }
  {
    float mx = 0.f;
    float lo[3] = {0, 0, 0}, hi[3] = {0, 0, 0};
    if (n > 0)
      for (int a = 0; a < 3; ++a) { lo[a] = o2f(h_scene[a]); hi[a] = o2f(h_scene[3 + a]); mx = fmaxf(mx, fmaxf(fabsf(lo[a]), fabsf(hi[a]))); }
    // Length tolerance: a few fp32 spacings of the largest coordinate (positions cannot be resolved finer).
    float eps_len = 4.0f * 1.1920929e-7f * mx;
    float tree_ms = 0.f, grid_ms = 0.f;
    cudaEventElapsedTime(&tree_ms, ev0, ev1);                                     // before the events are reused below
    c->bvh = DwBvh{c->d_nodes, c->d_tris, n_nodes, n, eps_len, nullptr, 0, make_float3(0, 0, 0), make_float3(0, 0, 0), make_float3(0, 0, 0),
                   nullptr, make_float3(0, 0, 0), make_float3(1, 1, 1)};
    rc = quantise_nodes(c, n_nodes, lo, hi, stream);
    if (rc != DW_OK) goto done;
    // ---- empty-space grid over the scene box (skipped for an empty or flat world)
    if (grid_req != -1) {
      rc = grid_build(c, n, tlo, thi, lo, hi, eps_len, GR, stream, &grid_built, &grid_free, &grid_ms);
      if (rc != DW_OK) goto done;
    }
    c->built = true;
    {   // the refit state takes over the boxes, the reference layout and the scene bounds
      dw_ctx::Refit& r = c->rf;
      r.n_refs = n; r.split_div = split_used; r.grid_res = grid_built;
      r.counts = counts; r.offs = offs; r.tlo = tlo_t; r.thi = thi_t; r.rlo = tlo; r.rhi = thi; r.scene = scene;
      counts = nullptr; offs = nullptr; tlo_t = nullptr; thi_t = nullptr; tlo = nullptr; thi = nullptr; scene = nullptr;
      r.level_start = levels;
      rc = nodes_area(c, n_nodes, stream, &r.build_area);
      if (rc != DW_OK) goto done;
    }
#if DW_WIDE8
    if (n > 0) {
      int n8 = 0;
      rc = widen8(c, n_nodes, stream, &n8);
      if (rc != DW_OK) goto done;
      n_nodes = n8;
      c->bvh.nodes = c->d_nodes; c->bvh.n_nodes = n8;
    }
#endif
    if (stats) {
      stats->n_tri = nt; stats->n_refs = n; stats->split_div = split_used; stats->n_nodes = n_nodes; stats->node_bytes = 128ll * n_nodes; stats->tri_bytes = 48ll * n;
      stats->max_depth = wide_depth; stats->n_leaves = h_misc[2];
      for (int a = 0; a < 3; ++a) { stats->scene_lo[a] = lo[a]; stats->scene_hi[a] = hi[a]; }
      stats->build_ms = tree_ms + grid_ms;
      stats->ploc_rounds = ploc_rounds; stats->binary_depth = h_misc[3];
      stats->grid_res = grid_built; stats->grid_free_cells = grid_free;
    }
  }
done:
  dw_sfree(tlo, stream); dw_sfree(thi, stream); dw_sfree(tlo_t, stream); dw_sfree(thi_t, stream); dw_sfree(counts, stream); dw_sfree(offs, stream); dw_sfree(ref_tri, stream); dw_sfree(blo, stream); dw_sfree(bhi, stream); dw_sfree(scene, stream); dw_sfree(keys, stream); dw_sfree(keys2, stream); dw_sfree(vals, stream);
  dw_sfree(vals2, stream); dw_sfree(left, stream); dw_sfree(right, stream); dw_sfree(parent, stream); dw_sfree(size, stream); dw_sfree(leftmost, stream); dw_sfree(nn, stream);
  dw_sfree(flag, stream); dw_sfree(bsum, stream); dw_sfree(boff, stream); dw_sfree(pst, stream); dw_sfree(slot, stream); dw_sfree(misc, stream); dw_sfree(tmp, stream); dw_sfree(nodes_tmp, stream); dw_sfree(occ, stream); dw_sfree(sat, stream);
  for (int k = 0; k < 2; ++k) { dw_sfree(cl[k], stream); dw_sfree(ch[k], stream); dw_sfree(cn[k], stream); dw_sfree(tasks[k], stream); }
  if (ev0) cudaEventDestroy(ev0);
  if (ev1) cudaEventDestroy(ev1);
  cudaStreamSynchronize(stream);   // the frees above are complete when the call returns: the next build finds its memory in the pool
  if (rc != DW_OK) dw_bvh_free(c);
  return rc;
}

// dw_refit_bvh: new vertex positions under the tree of the last build (include/darwinopt.h).
int dw_bvh_refit_impl(dw_ctx* c, const float* xyz, int on_device, dw_refit_stats* stats, cudaStream_t stream) {
  int rc = DW_OK;
  const int nt = (int)c->n_tri, B = 256;
  dw_ctx::Refit& r = c->rf;
  const int n = r.n_refs;
  unsigned long long* errs = nullptr;
  int* loose = nullptr;
  cudaEvent_t ev0 = nullptr, ev1 = nullptr;
  unsigned long long h_err[3] = {0, 0, ~0ull};
  unsigned h_scene[6] = {0, 0, 0, 0, 0, 0};
  int h_loose = 0, grid_built = 0, grid_free = 0;
  float lo[3] = {0, 0, 0}, hi[3] = {0, 0, 0}, mx = 0.f, eps_len = 0.f, ms = 0.f, grid_ms = 0.f;
  double area = 0.0;
  if (stats) { memset(stats, 0, sizeof *stats); stats->area_ratio = 1.0f; }
  if (nt == 0) return DW_OK;                                     // an empty world stays empty
  DW_B(cudaEventCreate(&ev0)); DW_B(cudaEventCreate(&ev1));
  DW_B(cudaMalloc(&errs, sizeof h_err)); DW_B(cudaMalloc(&loose, 4));
  DW_B(cudaEventRecord(ev0, stream));
  DW_B(cudaMemcpyAsync(c->d_xyz, xyz, sizeof(float) * 3 * (size_t)c->n_vert, on_device ? cudaMemcpyDeviceToDevice : cudaMemcpyHostToDevice, stream));
  DW_B(cudaMemcpyAsync(errs, h_err, sizeof h_err, cudaMemcpyHostToDevice, stream));
  DW_B(cudaMemsetAsync(loose, 0, 4, stream));
  {
    const unsigned init[6] = {0xffffffffu, 0xffffffffu, 0xffffffffu, 0u, 0u, 0u};
    DW_B(cudaMemcpyAsync(r.scene, init, sizeof init, cudaMemcpyHostToDevice, stream));
  }
  refit_check_kernel<<<G_blocks(nt, B), B, 0, stream>>>(nt, c->d_xyz, c->d_idx, errs);
  tri_bounds_kernel<<<G_blocks(nt, B), B, 0, stream>>>(nt, c->d_xyz, c->d_idx, r.tlo, r.thi, r.scene);
  DW_B(cudaMemcpyAsync(h_err, errs, sizeof h_err, cudaMemcpyDeviceToHost, stream));
  DW_B(cudaMemcpyAsync(h_scene, r.scene, sizeof h_scene, cudaMemcpyDeviceToHost, stream));
  DW_B(cudaStreamSynchronize(stream));
  if (h_err[0] || h_err[1]) {
    rc = dw_fail(c, DW_E_RANGE, "dw_refit_bvh: %llu triangles with non-finite vertices, %llu with zero area (first bad triangle %llu); "
                 "the geometry is no longer valid, set it again", h_err[0], h_err[1], h_err[2]);
    c->have_geom = false;
    goto done;
  }
  for (int a = 0; a < 3; ++a) { lo[a] = o2f(h_scene[a]); hi[a] = o2f(h_scene[3 + a]); mx = fmaxf(mx, fmaxf(fabsf(lo[a]), fabsf(hi[a]))); }
  eps_len = 4.0f * 1.1920929e-7f * mx;                           // as in the build: tolerance and padding follow the scene
  refit_refs_kernel<<<G_blocks(nt, B), B, 0, stream>>>(nt, c->d_xyz, c->d_idx, r.tlo, r.thi, r.scene, r.split_div, eps_len, r.offs, r.counts,
                                                       r.rlo, r.rhi, loose);
  refit_pack_kernel<<<G_blocks(n, B), B, 0, stream>>>(n, c->d_xyz, c->d_idx, c->d_tris);
  for (int k = (int)r.level_start.size() - 2; k >= 0; --k) {
    const int first = r.level_start[k], count = r.level_start[k + 1] - first;
    refit_level_kernel<<<G_blocks(count, B), B, 0, stream>>>(first, count, c->d_nodes, r.slot_ref, r.rlo, r.rhi);
  }
  DW_B(cudaGetLastError());
  DW_B(cudaMemcpyAsync(&h_loose, loose, 4, cudaMemcpyDeviceToHost, stream));
  c->bvh.eps_len = eps_len;
  if (r.grid_res > 0) {
    rc = grid_build(c, n, r.rlo, r.rhi, lo, hi, eps_len, r.grid_res, stream, &grid_built, &grid_free, &grid_ms);
    if (rc != DW_OK) goto done;
  }
  rc = quantise_nodes(c, c->bvh.n_nodes, lo, hi, stream);
  if (rc != DW_OK) goto done;
  rc = nodes_area(c, c->bvh.n_nodes, stream, &area);
  if (rc != DW_OK) goto done;
  DW_B(cudaEventRecord(ev1, stream));
  DW_B(cudaStreamSynchronize(stream));
  cudaEventElapsedTime(&ms, ev0, ev1);
  if (stats) {
    stats->area_ratio = r.build_area > 0.0 ? (float)(area / r.build_area) : 1.0f;
    stats->refit_ms = ms; stats->n_levels = (int)r.level_start.size() - 1; stats->n_loose_tris = h_loose; stats->grid_free_cells = grid_free;
    for (int a = 0; a < 3; ++a) { stats->scene_lo[a] = lo[a]; stats->scene_hi[a] = hi[a]; }
  }
done:
  cudaFree(errs); cudaFree(loose);
  if (ev0) cudaEventDestroy(ev0);
  if (ev1) cudaEventDestroy(ev1);
  if (rc != DW_OK) dw_bvh_free(c);
  return rc;
}
