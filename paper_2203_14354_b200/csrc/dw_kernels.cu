// dw_kernels.cu -- the hot path on the device: BVH first-hit query (S1) and the persistent-thread
// propagation kernel (S1..S13 of DESIGN.md; "photon propagation code", P:175 surface models,
// P:185-187 Fresnel/TIR checks, P:436-444 appendix fixes).  fp32 arithmetic throughout.
#include <float.h>
#include <math.h>

#include "dw_internal.cuh"

namespace {

constexpr float kInvC = 1.0f / 299.792458f;   // ns per mm in vacuum
constexpr int kStackShared = 12;              // per-thread traversal stack entries kept in shared memory
constexpr int kStackLocal = 64;               // overflow entries (local memory; only deep LBVH chains reach it)
constexpr float kEdgeSlack = 2e-6f;           // barycentric slack that closes fp32 cracks between triangles
constexpr float kBoxSlack = 1.0000005f;       // conservative slab test (robust traversal)

// ------------------------------------------------------------------------------------------------ RNG (S12)
// Philox4x32-10 (Salmon et al. 2011), key = seed, counter = (photon lo, photon hi, step, block).
__device__ __forceinline__ uint4 philox4x32_10(uint4 c, uint32_t k0, uint32_t k1) {
#pragma unroll
  for (int r = 0; r < 10; ++r) {
    uint32_t hi0 = __umulhi(0xD2511F53u, c.x), lo0 = 0xD2511F53u * c.x;
    uint32_t hi1 = __umulhi(0xCD9E8D57u, c.z), lo1 = 0xCD9E8D57u * c.z;
    c = make_uint4(hi1 ^ c.y ^ k0, lo1, hi0 ^ c.w ^ k1, lo0);
    k0 += 0x9E3779B9u;
    k1 += 0xBB67AE85u;
  }
  return c;
}
// ((x >> 9) + 0.5) * 2^-23: 24 significant bits, exact in fp32, strictly inside (0,1)
__device__ __forceinline__ float u01(uint32_t x) { return ((float)(x >> 9) + 0.5f) * 1.1920928955078125e-7f; }
__device__ __forceinline__ float4 draw4(uint64_t seed, uint64_t pid, uint32_t step, uint32_t block) {
  uint4 r = philox4x32_10(make_uint4((uint32_t)pid, (uint32_t)(pid >> 32), step, block), (uint32_t)seed, (uint32_t)(seed >> 32));
  return make_float4(u01(r.x), u01(r.y), u01(r.z), u01(r.w));
}

// ------------------------------------------------------------------------------------------------ vectors
struct V3 { float x, y, z; };
__device__ __forceinline__ V3 mk(float x, float y, float z) { V3 v; v.x = x; v.y = y; v.z = z; return v; }
__device__ __forceinline__ V3 operator+(V3 a, V3 b) { return mk(a.x + b.x, a.y + b.y, a.z + b.z); }
__device__ __forceinline__ V3 operator-(V3 a, V3 b) { return mk(a.x - b.x, a.y - b.y, a.z - b.z); }
__device__ __forceinline__ V3 operator*(float s, V3 a) { return mk(s * a.x, s * a.y, s * a.z); }
__device__ __forceinline__ float dot(V3 a, V3 b) { return fmaf(a.x, b.x, fmaf(a.y, b.y, a.z * b.z)); }
__device__ __forceinline__ V3 cross(V3 a, V3 b) {
  return mk(fmaf(a.y, b.z, -a.z * b.y), fmaf(a.z, b.x, -a.x * b.z), fmaf(a.x, b.y, -a.y * b.x));
}
__device__ __forceinline__ V3 unit(V3 a) { return rsqrtf(dot(a, a)) * a; }
__device__ __forceinline__ V3 fma3(float s, V3 a, V3 b) { return mk(fmaf(s, a.x, b.x), fmaf(s, a.y, b.y), fmaf(s, a.z, b.z)); }

// ------------------------------------------------------------------------------------------------ tables (S3)
__device__ __forceinline__ float table_at(const float* __restrict__ tab, int row, int nl, float l0, float inv_dl, float lambda) {
  const float* r = tab + (size_t)row * nl;
  if (nl == 1) return __ldg(r);
  float f = (lambda - l0) * inv_dl;
  if (!(f > 0.f)) return __ldg(r);
  if (f >= (float)(nl - 1)) return __ldg(r + nl - 1);
  int i = (int)f;
  float w = f - (float)i;
  float y0 = __ldg(r + i), y1 = __ldg(r + i + 1);
  if (isinf(y0) || isinf(y1)) return (w == 0.f) ? y0 : (isinf(y1) ? y1 : y0);
  return fmaf(w, y1 - y0, y0);
}

// ------------------------------------------------------------------------------------------------ first hit (S1)
struct Hit {
  float t;     // distance, +inf = none
  int slot;    // index into the leaf-ordered triangle array
  int id;      // caller triangle id
};

// Nearest triangle along o + t d with 0 < t < tmax, excluding caller id `exclude`; ties -> lowest caller id.
// medium >= 0: only triangles whose near side (the side the ray comes from) is `medium` count
// (DESIGN.md "medium culling"); medium < 0: every triangle counts (the definition S1).
// sstack: this thread's column of the shared-memory stack, entries `sstride` ints apart.
__device__ __forceinline__ Hit trace(const DwBvh& bvh, V3 o, V3 d, float tmax, int exclude, int medium, int* sstack,
                                     int sstride) {
  Hit best;
  best.t = tmax; best.slot = -1; best.id = 0x7fffffff;
  int lstack[kStackLocal];
  // inverse direction with zero components pushed to +-tiny so that 0 * inf never appears
  const float tiny = 1e-30f;
  V3 inv = mk(1.0f / (fabsf(d.x) > tiny ? d.x : copysignf(tiny, d.x)), 1.0f / (fabsf(d.y) > tiny ? d.y : copysignf(tiny, d.y)),
              1.0f / (fabsf(d.z) > tiny ? d.z : copysignf(tiny, d.z)));
  V3 oi = mk(o.x * inv.x, o.y * inv.y, o.z * inv.z);
  int sp = 0;
  int node = 0;
  const float4* __restrict__ nodes = bvh.nodes;
  const float4* __restrict__ tris = bvh.tris;
  while (true) {
    if (node >= 0) {
      if (node == DW_REF_NONE) goto pop;
      {
        const float4* p = nodes + 4 * (size_t)node;
        float4 q0 = __ldg(p), q1 = __ldg(p + 1), q2 = __ldg(p + 2), q3 = __ldg(p + 3);
        // child 0: lo (q0.x q0.y q0.z) hi (q0.w q1.x q1.y); child 1: lo (q1.z q1.w q2.x) hi (q2.y q2.z q2.w)
        float ax = fmaf(q0.x, inv.x, -oi.x), bx = fmaf(q0.w, inv.x, -oi.x);
        float ay = fmaf(q0.y, inv.y, -oi.y), by = fmaf(q1.x, inv.y, -oi.y);
        float az = fmaf(q0.z, inv.z, -oi.z), bz = fmaf(q1.y, inv.z, -oi.z);
        float n0 = fmaxf(fmaxf(fminf(ax, bx), fminf(ay, by)), fmaxf(fminf(az, bz), 0.f));
        float f0 = fminf(fminf(fmaxf(ax, bx), fmaxf(ay, by)), fminf(fmaxf(az, bz), best.t));
        ax = fmaf(q1.z, inv.x, -oi.x); bx = fmaf(q2.y, inv.x, -oi.x);
        ay = fmaf(q1.w, inv.y, -oi.y); by = fmaf(q2.z, inv.y, -oi.y);
        az = fmaf(q2.x, inv.z, -oi.z); bz = fmaf(q2.w, inv.z, -oi.z);
        float n1 = fmaxf(fmaxf(fminf(ax, bx), fminf(ay, by)), fmaxf(fminf(az, bz), 0.f));
        float f1 = fminf(fminf(fmaxf(ax, bx), fmaxf(ay, by)), fminf(fmaxf(az, bz), best.t));
        int r0 = __float_as_int(q3.x), r1 = __float_as_int(q3.y);
        bool h0 = (n0 <= fmaf(f0, kBoxSlack, bvh.eps_len)) && (r0 != DW_REF_NONE);
        bool h1 = (n1 <= fmaf(f1, kBoxSlack, bvh.eps_len)) && (r1 != DW_REF_NONE);
        if (h0 && h1) {
          int nearr = r0, farr = r1;
          if (n1 < n0) { nearr = r1; farr = r0; }
          if (sp < kStackShared) sstack[sp * sstride] = farr; else lstack[sp - kStackShared] = farr;
          ++sp;
          node = nearr;
          continue;
        }
        if (h0) { node = r0; continue; }
        if (h1) { node = r1; continue; }
        goto pop;
      }
    } else {
      // leaf: ~node = (first << 3) | (count - 1)
      int code = ~node;
      int first = code >> 3, cnt = (code & 7) + 1;
      for (int i = 0; i < cnt; ++i) {
        const float4* p = tris + 3 * (size_t)(first + i);
        float4 a = __ldg(p), b = __ldg(p + 1), c = __ldg(p + 2);
        V3 e1 = mk(a.w, b.x, b.y), e2 = mk(b.z, b.w, c.x);
        V3 pv = cross(d, e2);
        float det = dot(e1, pv);
        if (fabsf(det) < 1e-30f) continue;
        float idet = 1.0f / det;
        V3 tv = mk(o.x - a.x, o.y - a.y, o.z - a.z);
        float u = dot(tv, pv) * idet;
        V3 qv = cross(tv, e1);
        float v = dot(d, qv) * idet;
        float t = dot(e2, qv) * idet;
        int id = __float_as_int(c.y);
        bool ok = (u >= -kEdgeSlack) && (v >= -kEdgeSlack) && (u + v <= 1.0f + kEdgeSlack) && (t > 0.f) &&
                  (t < best.t || (t == best.t && id < best.id)) && (id != exclude);
        if (ok && medium >= 0) {
          uint32_t cw = __float_as_uint(c.z);
          int near_side = (det > 0.f) ? (int)((cw >> 8) & 0xFF) : (int)(cw & 0xFF);   // det > 0: ray comes from the outer side
          ok = (near_side == medium);
        }
        if (ok) { best.t = t; best.slot = first + i; best.id = id; }
      }
    }
  pop:
    if (sp == 0) break;
    --sp;
    node = (sp < kStackShared) ? sstack[sp * sstride] : lstack[sp - kStackShared];
  }
  if (best.slot < 0) best.t = INFINITY;
  return best;
}

__global__ void __launch_bounds__(128) first_hit_kernel(DwBvh bvh, int64_t n, const float* __restrict__ ox,
                                                        const float* __restrict__ oy, const float* __restrict__ oz,
                                                        const float* __restrict__ dx, const float* __restrict__ dy,
                                                        const float* __restrict__ dz, const int32_t* __restrict__ exclude,
                                                        int32_t* __restrict__ tri, float* __restrict__ dist) {
  extern __shared__ int s_stack[];
  int64_t i = blockIdx.x * (int64_t)blockDim.x + threadIdx.x;
  if (i >= n) return;
  Hit h = trace(bvh, mk(ox[i], oy[i], oz[i]), mk(dx[i], dy[i], dz[i]), INFINITY, exclude ? exclude[i] : -1, -1,
                s_stack + threadIdx.x, blockDim.x);
  tri[i] = h.slot >= 0 ? h.id : -1;
  dist[i] = h.t;
}

// ------------------------------------------------------------------------------------------------ physics
// tangent frame about a unit vector w (S7): a = normalize(ref x w), b = w x a, ref = x if |w.x| < 0.5 else y
__device__ __forceinline__ void frame(V3 w, V3& a, V3& b) {
  V3 ref = (fabsf(w.x) < 0.5f) ? mk(1.f, 0.f, 0.f) : mk(0.f, 1.f, 0.f);
  a = unit(cross(ref, w));
  b = cross(w, a);
}

// S6 Rayleigh scattering: the algorithm that reproduces the theoretical distribution:
// isotropic k', accept with probability |e - (e.k')k'|^2; iteration j uses Philox block 1 + j.
__device__ __forceinline__ bool rayleigh(V3& k, V3& e, uint64_t seed, uint64_t pid, uint32_t step) {
  for (uint32_t j = 0; j < 4096u; ++j) {
    float4 r = draw4(seed, pid, step, 1u + j);
    float ct = 1.0f - 2.0f * r.x;
    float st = sqrtf(fmaxf(0.f, 1.0f - ct * ct));
    float sp, cp;
    sincospif(2.0f * r.y, &sp, &cp);
    V3 kn = mk(st * cp, st * sp, ct);
    V3 er = fma3(-dot(e, kn), kn, e);
    float w = dot(er, er);
    if (r.z < w) { k = kn; e = rsqrtf(w) * er; return true; }
  }
  return false;
}

// S7 diffuse reflection (Lambert): block 1 = (cos^2 theta, azimuth, polarisation angle, -)
__device__ __forceinline__ void lambert(V3 nh, V3& k, V3& e, float4 r) {
  float ct = sqrtf(r.x), st = sqrtf(fmaxf(0.f, 1.0f - r.x));
  float sp, cp;
  sincospif(2.0f * r.y, &sp, &cp);
  V3 a, b;
  frame(nh, a, b);
  k = unit(fma3(ct, nh, fma3(st * cp, a, (st * sp) * b)));
  sincospif(2.0f * r.z, &sp, &cp);
  frame(k, a, b);
  e = fma3(cp, a, sp * b);
}

// S8 Fresnel; nh faces the photon.  Returns history bits.
__device__ __forceinline__ uint32_t fresnel(float n1, float n2, V3 nh, V3& k, V3& e, float u, bool& crossed) {
  float ci = -dot(k, nh);
  V3 sv = cross(k, nh);
  float si2 = dot(sv, sv);
  float si = sqrtf(si2);
  V3 s; float Es, Ep;
  if (si < 1e-5f) { s = e; Es = 1.f; Ep = 0.f; }           // normal incidence must never abort
  else { s = (1.0f / si) * sv; V3 p = cross(s, k); Es = dot(e, s); Ep = dot(e, p); }
  float eta = n1 / n2;
  float st = eta * si;
  crossed = false;
  if (st >= 1.0f) {                                          // total internal reflection
    V3 kr = unit(fma3(2.0f * ci, nh, k));
    e = unit(fma3(Es, s, Ep * cross(s, kr)));
    k = kr;
    return DW_H_FRESNEL_REFLECT | DW_H_TIR;
  }
  float ct = sqrtf(fmaxf(0.f, 1.0f - st * st));
  float a = n1 * ci, b = n2 * ct, c2 = n2 * ci, d2 = n1 * ct;
  float rs = (a - b) / (a + b), rp = (c2 - d2) / (c2 + d2);
  float R = Es * Es * rs * rs + Ep * Ep * rp * rp;
  if (u < R) {
    V3 kr = unit(fma3(2.0f * ci, nh, k));
    e = unit(fma3(rs * Es, s, (rp * Ep) * cross(s, kr)));
    k = kr;
    return DW_H_FRESNEL_REFLECT;
  }
  float ts = 2.0f * a / (a + b), tp = 2.0f * a / (c2 + d2);
  V3 kt = unit(fma3(eta, k, (eta * ci - ct) * nh));
  e = unit(fma3(ts * Es, s, (tp * Ep) * cross(s, kt)));
  k = kt;
  crossed = true;
  return DW_H_FRESNEL_REFRACT;
}

// ------------------------------------------------------------------------------------------------ propagation
struct PropArgs {
  DwBvh bvh;
  DwTables tab;
  dw_photons in;
  dw_results out;
  dw_hists hist;
  uint64_t seed;
  int32_t max_steps;
  uint32_t flags;
  unsigned long long* queue_head;   // device counter, zeroed before launch
};

constexpr int kChunk = 8;   // photons claimed per lane per queue transaction (x32 per warp)

__global__ void __launch_bounds__(128, 6) propagate_kernel(const __grid_constant__ PropArgs A) {
  extern __shared__ int s_stack[];
  __shared__ unsigned int s_fate[8];
  __shared__ unsigned long long s_steps;
  if (threadIdx.x < 8) s_fate[threadIdx.x] = 0;
  if (threadIdx.x == 0) s_steps = 0ull;
  __syncthreads();
  int* my_stack = s_stack + threadIdx.x;
  const int sstride = blockDim.x;
  const int lane = threadIdx.x & 31;
  const int64_t n = A.in.n;
  const bool literal = (A.flags & DW_PROP_UNBOUNDED_QUERY) != 0;

  // warp-private range of photon indices [w_next, w_end)
  int64_t w_next = 0, w_end = 0;
  bool active = false;
  // photon state
  int64_t pi = 0;
  V3 x = mk(0, 0, 0), k = mk(0, 0, 1), e = mk(1, 0, 0);
  float lambda = 0.f, t = 0.f;
  int medium = -1, last_tri = -1;
  uint32_t step = 0, hist = 0;

  while (true) {
    // ---------------------------------------------------------------- a2: refill finished lanes
    unsigned idle = __ballot_sync(0xffffffffu, !active);
    if (idle) {
      int need = __popc(idle);
      if (w_end - w_next < need && w_end >= 0) {           // claim a new chunk for the warp (one atomic per warp)
        // keep what is left of the old chunk only if it is empty (ranges are consumed in order, so the remainder
        // is always used up before a new claim is needed); w_end < 0 marks "queue exhausted"
        if (w_next == w_end) {
          unsigned long long base = 0;
          if (lane == 0) base = atomicAdd(A.queue_head, (unsigned long long)(32 * kChunk));
          base = __shfl_sync(0xffffffffu, base, 0);
          w_next = (int64_t)base;
          w_end = (int64_t)base + 32 * kChunk;
          if (w_next >= n) { w_next = 0; w_end = -1; }
          else if (w_end > n) w_end = n;
        }
      }
      if (w_end > w_next) {
        int rank = __popc(idle & ((1u << lane) - 1u));
        int avail = (int)min((int64_t)need, w_end - w_next);
        if (!active && rank < avail) {
          pi = w_next + rank;
          x = mk(A.in.px[pi], A.in.py[pi], A.in.pz[pi]);
          k = mk(A.in.kx[pi], A.in.ky[pi], A.in.kz[pi]);
          e = mk(A.in.ex[pi], A.in.ey[pi], A.in.ez[pi]);
          lambda = A.in.wavelength[pi];
          t = A.in.t0[pi];
          medium = -1; last_tri = -1; step = 0; hist = 0;
          active = true;
        }
        w_next += avail;
      }
      if (__ballot_sync(0xffffffffu, active) == 0u) {
        if (w_end < 0) break;        // nothing running and the queue is exhausted
        continue;                    // chunk boundary: claim again
      }
    }

    // ---------------------------------------------------------------- one step of the loop S1..S11
    uint32_t fate = 0xFFu;           // 0xFF = still running
    int channel = -1;
    if (active) {
      const uint64_t pid = A.in.photon_id_base + (uint64_t)pi;
      if ((int32_t)step >= A.max_steps) {
        fate = DW_FATE_TRUNCATED;                                     // S10
      } else if (!(isfinite(x.x + x.y + x.z) && isfinite(k.x + k.y + k.z) && isfinite(e.x + e.y + e.z) && isfinite(t))) {
        fate = DW_FATE_NAN_ABORT;                                     // S11
      } else {
        float4 r0 = draw4(A.seed, pid, step, 0u);                     // (u_a, u_s, u_surface, u_fresnel)
        float n1 = 1.f, dbulk = INFINITY;
        bool absorb_first = false;
        bool bounded = (!literal) && (medium >= 0);
        if (bounded) {                                                // medium known: S3/S4 draws before the query
          n1 = table_at(A.tab.mat, medium, A.tab.nl_mat, A.tab.mat_l0, A.tab.mat_inv_dl, lambda);
          float La = table_at(A.tab.mat + (size_t)A.tab.n_mat * A.tab.nl_mat, medium, A.tab.nl_mat, A.tab.mat_l0, A.tab.mat_inv_dl, lambda);
          float Ls = table_at(A.tab.mat + 2 * (size_t)A.tab.n_mat * A.tab.nl_mat, medium, A.tab.nl_mat, A.tab.mat_l0, A.tab.mat_inv_dl, lambda);
          float da = -La * logf(r0.x), ds = -Ls * logf(r0.y);
          absorb_first = da < ds;
          dbulk = fminf(da, ds);
        }
        Hit h = trace(A.bvh, x, k, bounded ? dbulk + A.bvh.eps_len : INFINITY, last_tri, bounded ? medium : -1, my_stack, sstride);
        float4 tc = make_float4(0, 0, 0, 0), ta = tc, tb = tc;
        int m1 = medium, m2 = medium;
        V3 ng = mk(0, 0, 1);
        bool toward_outer = false;
        if (h.slot >= 0) {                                            // S2 sides
          const float4* p = A.bvh.tris + 3 * (size_t)h.slot;
          ta = __ldg(p); tb = __ldg(p + 1); tc = __ldg(p + 2);
          ng = unit(cross(mk(ta.w, tb.x, tb.y), mk(tb.z, tb.w, tc.x)));
          uint32_t cw = __float_as_uint(tc.z);
          toward_outer = dot(k, ng) > 0.f;
          int mi = (int)(cw & 0xFF), mo = (int)((cw >> 8) & 0xFF);
          m1 = toward_outer ? mi : mo;
          m2 = toward_outer ? mo : mi;
        }
        if (!bounded) {
          if (h.slot < 0) {
            fate = DW_FATE_ESCAPED;                                   // G3: ray leaves the world
          } else {
            if (medium >= 0 && medium != m1) hist |= DW_H_MEDIUM_MISMATCH;
            medium = m1;
            n1 = table_at(A.tab.mat, m1, A.tab.nl_mat, A.tab.mat_l0, A.tab.mat_inv_dl, lambda);
            float La = table_at(A.tab.mat + (size_t)A.tab.n_mat * A.tab.nl_mat, m1, A.tab.nl_mat, A.tab.mat_l0, A.tab.mat_inv_dl, lambda);
            float Ls = table_at(A.tab.mat + 2 * (size_t)A.tab.n_mat * A.tab.nl_mat, m1, A.tab.nl_mat, A.tab.mat_l0, A.tab.mat_inv_dl, lambda);
            float da = -La * logf(r0.x), ds = -Ls * logf(r0.y);
            absorb_first = da < ds;
            dbulk = fminf(da, ds);
          }
        }
        if (fate == 0xFFu) {
          bool surface_event = (h.slot >= 0) && (bounded ? true : !(dbulk < h.t));
          if (!surface_event) {
            if (!(dbulk < INFINITY)) {
              fate = DW_FATE_ESCAPED;                                 // bounded query, no bulk process, nothing hit
            } else {
              x = fma3(dbulk, k, x);
              t = fmaf(dbulk * n1, kInvC, t);
              if (absorb_first) {
                fate = DW_FATE_BULK_ABSORBED;                         // S4 first branch
              } else {                                                // S4 second branch + S6
                if (!rayleigh(k, e, A.seed, pid, step)) fate = DW_FATE_NAN_ABORT;
                hist |= DW_H_RAYLEIGH;
                last_tri = -1;
              }
            }
          } else {                                                    // S4 third branch, S5
            x = fma3(h.t, k, x);
            t = fmaf(h.t * n1, kInvC, t);
            last_tri = h.id;
            if (medium != m1) hist |= DW_H_MEDIUM_MISMATCH;
            V3 nh = toward_outer ? mk(-ng.x, -ng.y, -ng.z) : ng;
            uint32_t cw = __float_as_uint(tc.z);
            int sf = (int)((cw >> 16) & 0xFF);
            if (sf != 0xFF) {                                         // S7 explicit surface
              const size_t ss = (size_t)A.tab.n_surf * A.tab.nl_surf;
              float c0 = table_at(A.tab.surf, sf, A.tab.nl_surf, A.tab.surf_l0, A.tab.surf_inv_dl, lambda);
              float c1 = table_at(A.tab.surf + ss, sf, A.tab.nl_surf, A.tab.surf_l0, A.tab.surf_inv_dl, lambda);
              float c2 = table_at(A.tab.surf + 2 * ss, sf, A.tab.nl_surf, A.tab.surf_l0, A.tab.surf_inv_dl, lambda);
              float c3 = table_at(A.tab.surf + 3 * ss, sf, A.tab.nl_surf, A.tab.surf_l0, A.tab.surf_inv_dl, lambda);
              float u = r0.z;
              if (u < c0) { fate = DW_FATE_DETECTED; channel = __float_as_int(tc.w); }
              else if (u < c1) { lambert(nh, k, e, draw4(A.seed, pid, step, 1u)); hist |= DW_H_REFLECT_DIFFUSE; }
              else if (u < c2) {                                      // specular: no plane of incidence needed
                k = unit(fma3(-2.0f * dot(k, nh), nh, k));
                e = unit(fma3(-2.0f * dot(e, nh), nh, e));
                hist |= DW_H_REFLECT_SPECULAR;
              }
              else if (u < c3) { hist |= DW_H_SURFACE_TRANSMIT; medium = m2; }
              else fate = DW_FATE_SURFACE_ABSORBED;
            } else {                                                  // S8 Fresnel
              float n2 = table_at(A.tab.mat, m2, A.tab.nl_mat, A.tab.mat_l0, A.tab.mat_inv_dl, lambda);
              bool crossed;
              hist |= fresnel(n1, n2, nh, k, e, r0.w, crossed);
              if (crossed) medium = m2;
            }
          }
          ++step;                                                     // S9 (the terminating iteration counts, S13)
        }
      }
    }

    // ---------------------------------------------------------------- a10: outputs and reductions
    if (fate != 0xFFu) {
      if (A.out.flags) A.out.flags[pi] = fate | hist;
      if (A.out.channel) A.out.channel[pi] = channel;
      if (A.out.t) A.out.t[pi] = t;
      if (A.out.steps) A.out.steps[pi] = step;
      if (A.out.last_tri) A.out.last_tri[pi] = last_tri;
      if (A.out.x) A.out.x[pi] = x.x;
      if (A.out.y) A.out.y[pi] = x.y;
      if (A.out.z) A.out.z[pi] = x.z;
      if (A.out.kx) { A.out.kx[pi] = k.x; A.out.ky[pi] = k.y; A.out.kz[pi] = k.z; }
      if (A.out.ex) { A.out.ex[pi] = e.x; A.out.ey[pi] = e.y; A.out.ez[pi] = e.z; }
      atomicAdd(&s_fate[fate & 7u], 1u);
      atomicAdd(&s_steps, (unsigned long long)step);
      active = false;
    }
    // detected photons: per-channel counts and arrival-time histogram, aggregated over equal keys in the warp
    unsigned det = __ballot_sync(0xffffffffu, fate == DW_FATE_DETECTED);
    if (det) {
      bool mine = fate == DW_FATE_DETECTED;
      if (A.hist.chan_count) {
        bool ok = mine && channel >= 0 && channel < A.hist.n_chan;
        unsigned peers = __match_any_sync(0xffffffffu, ok ? channel : -1 - lane);
        if (ok && lane == (__ffs(peers) - 1)) atomicAdd((unsigned long long*)&A.hist.chan_count[channel], (unsigned long long)__popc(peers));
      }
      if (A.hist.time_hist && A.hist.n_bins > 0) {
        float fb = floorf((t - A.hist.t_min) / A.hist.dt);
        int bin = fb < 0.f ? 0 : (fb > (float)(A.hist.n_bins - 1) ? (int)(A.hist.n_bins - 1) : (int)fb);
        unsigned peers = __match_any_sync(0xffffffffu, mine ? bin : -1 - lane);
        if (mine && lane == (__ffs(peers) - 1)) atomicAdd(&A.hist.time_hist[bin], (unsigned)__popc(peers));
      }
    }
  }

  __syncthreads();
  if (threadIdx.x < 8 && A.hist.fate_count && s_fate[threadIdx.x]) atomicAdd((unsigned long long*)&A.hist.fate_count[threadIdx.x], (unsigned long long)s_fate[threadIdx.x]);
  if (threadIdx.x == 0 && A.hist.total_steps && s_steps) atomicAdd((unsigned long long*)A.hist.total_steps, s_steps);
}

__global__ void philox_debug_kernel(uint64_t seed, uint64_t base, uint32_t step, uint32_t block, int64_t n,
                                    uint32_t* __restrict__ out_raw, float* __restrict__ out_u) {
  int64_t i = blockIdx.x * (int64_t)blockDim.x + threadIdx.x;
  if (i >= n) return;
  uint64_t pid = base + (uint64_t)i;
  uint4 r = philox4x32_10(make_uint4((uint32_t)pid, (uint32_t)(pid >> 32), step, block), (uint32_t)seed, (uint32_t)(seed >> 32));
  if (out_raw) { out_raw[4 * i] = r.x; out_raw[4 * i + 1] = r.y; out_raw[4 * i + 2] = r.z; out_raw[4 * i + 3] = r.w; }
  if (out_u) { out_u[4 * i] = u01(r.x); out_u[4 * i + 1] = u01(r.y); out_u[4 * i + 2] = u01(r.z); out_u[4 * i + 3] = u01(r.w); }
}

}  // namespace

int dw_first_hit_impl(dw_ctx* c, int64_t n, const float* ox, const float* oy, const float* oz, const float* dx,
                      const float* dy, const float* dz, const int32_t* exclude, int32_t* tri, float* dist, cudaStream_t stream) {
  const int B = 128;
  size_t smem = sizeof(int) * kStackShared * B;
  first_hit_kernel<<<(unsigned)((n + B - 1) / B), B, smem, stream>>>(c->bvh, n, ox, oy, oz, dx, dy, dz, exclude, tri, dist);
  DW_CUDA(c, cudaGetLastError());
  return DW_OK;
}

int dw_propagate_impl(dw_ctx* c, const dw_photons* in, uint64_t seed, int32_t max_steps, const dw_results* out,
                      const dw_hists* hist, const dw_propagate_params* params, cudaStream_t stream) {
  static_assert(sizeof(PropArgs) <= 4000, "kernel parameter block too large");
  PropArgs A{};
  A.bvh = c->bvh; A.tab = c->tables; A.in = *in;
  if (out) A.out = *out;
  if (hist) A.hist = *hist;
  A.seed = seed; A.max_steps = max_steps; A.flags = params ? params->flags : 0u;
  int B = (params && params->block_threads) ? params->block_threads : 128;
  if (B < 32 || B > 128 || (B & 31)) return dw_fail(c, DW_E_ARG, "dw_propagate: block_threads must be 32, 64, 96 or 128");
  size_t smem = sizeof(int) * kStackShared * B;
  int per_sm = 0;
  DW_CUDA(c, cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, propagate_kernel, B, smem));
  if (params && params->blocks_per_sm > 0) per_sm = std::min(per_sm, params->blocks_per_sm);
  if (per_sm < 1) return dw_fail(c, DW_E_CUDA, "dw_propagate: kernel does not fit on an SM");
  int64_t warps_needed = (in->n + 31) / 32;
  int64_t blocks_needed = (warps_needed + (B / 32) - 1) / (B / 32);
  int grid = (int)std::min<int64_t>((int64_t)c->sm_count * per_sm, std::max<int64_t>(blocks_needed, 1));
  // queue head lives in a small device allocation owned by the context-less stream-ordered pool
  unsigned long long* head = nullptr;
  DW_CUDA(c, cudaMallocAsync((void**)&head, sizeof(unsigned long long), stream));
  DW_CUDA(c, cudaMemsetAsync(head, 0, sizeof(unsigned long long), stream));
  A.queue_head = head;
  propagate_kernel<<<grid, B, smem, stream>>>(A);
  cudaError_t e = cudaGetLastError();
  cudaFreeAsync(head, stream);
  if (e != cudaSuccess) return dw_fail(c, DW_E_CUDA, "propagate_kernel launch failed: %s", cudaGetErrorString(e));
  c->last_grid = grid; c->last_block = B; c->last_smem = (int)smem; c->n_launches += 1;
  return DW_OK;
}

int dw_debug_philox_impl(dw_ctx* c, uint64_t seed, uint64_t base, uint32_t step, uint32_t block, int64_t n,
                         uint32_t* out_raw, float* out_u, cudaStream_t stream) {
  philox_debug_kernel<<<(unsigned)((n + 255) / 256), 256, 0, stream>>>(seed, base, step, block, n, out_raw, out_u);
  DW_CUDA(c, cudaGetLastError());
  return DW_OK;
}
