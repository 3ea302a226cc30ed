// dw_kernels.cu -- the hot path on the device: BVH first-hit query (S1) and the persistent-thread
// propagation kernel (S1..S13 of DESIGN.md; "photon propagation code", P:175 surface models,
// P:185-187 Fresnel/TIR checks, P:436-444 appendix fixes).  fp32 arithmetic throughout.
#include <float.h>
#include <stddef.h>
#include <math.h>

#include "dw_internal.cuh"

namespace {

// Node planes read as four 256-bit loads instead of seven 128-bit ones.  Neutral while the kernel was bound by instruction issue (199.1 vs
// 199.0); once Philox and the votes were cheaper the L1 data pipe (82 % busy, 97 % of its global wavefronts = lanes x node loads) was
// the limit: C2 227.2 -> 232.8, C3 211.4 -> 220.7 M photons/s (profiles/r01_captures_9_to_12_c2.md).
#ifndef DW_NODE_LDG256
#define DW_NODE_LDG256 1
#endif
#ifndef DW_FLAT_TABLES
#define DW_FLAT_TABLES 1
#endif
// Inlining of helpers that are called from many places (profiles/r01_propagate_bvh4_c2.md, capture 6: instruction fetch
// became the largest stall once the kernel grew to ~2900 instructions).  Level 0: everything inline; 1: Philox out of line;
// 2: + table look-up; 3: + Rayleigh / Lambert / Fresnel.
// Measured on C2 (alternating A/B, two rounds): level 0 173.8, 1 175.2, 2 188.6, 3 151.0 M photons/s.
// The pool kernel has since stopped calling either helper (flat tables, draw4_keys inlined: profiles/r01_captures_9_to_12_c2.md); the legacy
// kernel and dw_emit still do.
#ifndef DW_OUTLINE
#define DW_OUTLINE 2
#endif
#if DW_OUTLINE >= 1
#define DW_INL_PHILOX __noinline__
#else
#define DW_INL_PHILOX __forceinline__
#endif
#if DW_OUTLINE >= 2
#define DW_INL_TABLE __noinline__
#else
#define DW_INL_TABLE __forceinline__
#endif
#if DW_OUTLINE >= 3
#define DW_INL_PHYS __noinline__
#else
#define DW_INL_PHYS __forceinline__
#endif

constexpr float kInvC = 1.0f / 299.792458f;   // ns per mm in vacuum
constexpr int kStackShared = kDwStackShared;  // per-thread traversal stack entries kept in shared memory
constexpr int kStackLocal = kDwStackLocal;    // overflow entries (local memory; only unusually deep trees reach it)
#ifndef DW_SEAM_BACK
#define DW_SEAM_BACK 1
#endif
#ifndef DW_EDGE_REFINE
#define DW_EDGE_REFINE 1
#endif
constexpr int kThruSlack = 0x40000000;
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
#ifndef DW_U01_FMA
#define DW_U01_FMA 1
#endif
#if DW_U01_FMA   // one FMA: (x >> 9) < 2^23, so f * 2^-23 + 2^-24 is exact and equals the expression above bit for bit
__device__ __forceinline__ float u01(uint32_t x) { return fmaf((float)(x >> 9), 1.1920928955078125e-7f, 5.9604644775390625e-8f); }
#else
__device__ __forceinline__ float u01(uint32_t x) { return ((float)(x >> 9) + 0.5f) * 1.1920928955078125e-7f; }
#endif
__device__ DW_INL_PHILOX float4 draw4(uint64_t seed, uint64_t pid, uint32_t step, uint32_t block) {
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
__device__ DW_INL_TABLE float table_at(const float* __restrict__ tab, int row, int nl, float l0, float inv_dl, float lambda) {
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
// The query is written as a resumable state machine so that the propagation kernel can interleave the
// traversal steps of all lanes of a warp; dw_first_hit runs it to completion.
// DW_NODE_Q16 (dw_internal.cuh): 64-byte nodes with 16-bit planes (DwBvh::qnodes) instead of the 128-byte fp32 nodes
struct Ray {
  V3 o, d;     // origin, unit direction
  V3 inv, oi;  // fp32 nodes: 1/d (zero components pushed to +-1e30) and o * inv, so that a plane p is met at p * inv - oi;
               // 16-bit nodes: the same for a plane given as q steps of q_cs from q_lo: q * (q_cs / d) - (o - q_lo) / d
};
// 1 / det of the triangle test by MUFU as well: another 0.8 %, but the finer closed sphere then leaks 6 of 4e6 photons instead of 2
// (budget 4: tests/test_gpu_parity.py test_leak_budget_second_seed_and_finer_sphere); the edge rules count on the rounded quotient.  Off.
#ifndef DW_TRI_RCP_APPROX
#define DW_TRI_RCP_APPROX 0
#endif
// 1 / d of the ray set-up by MUFU.RCP alone (C2 42.18 -> 41.67 ms, C3 44.44 -> 43.93; results unchanged on C0-C3, 86 GPU tests pass).
#ifndef DW_RAY_RCP_APPROX
#define DW_RAY_RCP_APPROX 1
#endif
__device__ __forceinline__ float rcp_approx(float x) { float y; asm("rcp.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x)); return y; }
__device__ __forceinline__ void ray_setup(Ray& r, V3 o, V3 d, const DwBvh& bvh) {
  const float tiny = 1e-30f;   // zero components become +-tiny so that 0 * inf never appears
  r.o = o; r.d = d;
#if DW_RAY_RCP_APPROX   // one MUFU each (1 ulp; the slab test has a slack of 8 ulp): an IEEE division is 14 instructions with its slow path
  const V3 inv = mk(rcp_approx(fabsf(d.x) > tiny ? d.x : copysignf(tiny, d.x)), rcp_approx(fabsf(d.y) > tiny ? d.y : copysignf(tiny, d.y)),
                    rcp_approx(fabsf(d.z) > tiny ? d.z : copysignf(tiny, d.z)));
#else
  const V3 inv = mk(1.0f / (fabsf(d.x) > tiny ? d.x : copysignf(tiny, d.x)), 1.0f / (fabsf(d.y) > tiny ? d.y : copysignf(tiny, d.y)),
                    1.0f / (fabsf(d.z) > tiny ? d.z : copysignf(tiny, d.z)));
#endif
#if DW_NODE_Q16
  r.inv = mk(bvh.q_cs.x * inv.x, bvh.q_cs.y * inv.y, bvh.q_cs.z * inv.z);
  r.oi = mk((o.x - bvh.q_lo.x) * inv.x, (o.y - bvh.q_lo.y) * inv.y, (o.z - bvh.q_lo.z) * inv.z);
#else
  r.inv = inv;
  r.oi = mk(o.x * inv.x, o.y * inv.y, o.z * inv.z);
#endif
}

constexpr int kInLeaf = -1;   // TraceState::node: triangles [tri_cur, tri_end) are pending
constexpr int kDone = -2;     // TraceState::node: traversal finished
struct TraceState {
  int node;                   // >= 0: internal node to visit next
  int sp;                     // stack depth
  int tri_cur, tri_end;       // pending triangle slots of the current leaf
  float best_t;               // nearest accepted distance so far (starts at t_max)
  int best_slot, best_id;     // leaf-order slot and caller id of the nearest triangle (-1 / INT_MAX: none); bit 30 of best_id
                              // (kThruSlack): that triangle was accepted through the edge slack only (ids are < 2^28)
};
__device__ __forceinline__ void ts_begin(TraceState& s, float tmax) {
  s.node = 0; s.sp = 0; s.tri_cur = 0; s.tri_end = 0; s.best_t = tmax; s.best_slot = -1; s.best_id = 0x7fffffff;
}
// Continue with child reference `ref` (>= 0 internal, < 0 leaf) or, for DW_REF_NONE, with the stack top.
__device__ __forceinline__ void ts_goto(TraceState& s, int ref, const int* sstack, int sstride, const int* lstack) {
  if (ref == DW_REF_NONE) {
    if (s.sp == 0) { s.node = kDone; return; }
    --s.sp;
    ref = (s.sp < kStackShared) ? sstack[s.sp * sstride] : lstack[s.sp - kStackShared];
  }
  if (ref >= 0) { s.node = ref; return; }
  int code = ~ref;                       // leaf: (first << 3) | (count - 1)
  s.tri_cur = code >> 3;
  s.tri_end = (code >> 3) + (code & 7) + 1;
  s.node = kInLeaf;
}

// One 4-wide node: slab-test the four children against [0, best_t]; the nearest hit is visited next, the others are
// pushed.  Empty children carry DW_REF_NONE (their inverted boxes alone would not reject: inf arithmetic).
__device__ __forceinline__ bool slab(const Ray& r, float best_t, float eps, float lox, float loy, float loz, float hix,
                                     float hiy, float hiz, float& tnear) {
  float ax = fmaf(lox, r.inv.x, -r.oi.x), bx = fmaf(hix, r.inv.x, -r.oi.x);
  float ay = fmaf(loy, r.inv.y, -r.oi.y), by = fmaf(hiy, r.inv.y, -r.oi.y);
  float az = fmaf(loz, r.inv.z, -r.oi.z), bz = fmaf(hiz, r.inv.z, -r.oi.z);
  tnear = fmaxf(fmaxf(fminf(ax, bx), fminf(ay, by)), fmaxf(fminf(az, bz), 0.f));
  float tfar = fminf(fminf(fmaxf(ax, bx), fmaxf(ay, by)), fminf(fmaxf(az, bz), best_t));
  return tnear <= fmaf(tfar, kBoxSlack, eps);
}
__device__ __forceinline__ void ts_push(TraceState& s, int ref, int* sstack, int sstride, int* lstack) {
  if (s.sp < kStackShared) sstack[s.sp * sstride] = ref; else lstack[s.sp - kStackShared] = ref;
  ++s.sp;
}
// 256-bit read-only load (sm_100: LDG.E.256): a node visit is 4 load instructions instead of 7, and the L1 cost of a divergent
// load is paid per instruction and line (profiles/r01_final_c2.md: L1 throughput is the nearest limit).  p must be 32-byte aligned.
__device__ __forceinline__ void ldg256(const float4* p, float4& a, float4& b) {
  asm volatile("ld.global.nc.v8.f32 {%0,%1,%2,%3,%4,%5,%6,%7}, [%8];"
               : "=f"(a.x), "=f"(a.y), "=f"(a.z), "=f"(a.w), "=f"(b.x), "=f"(b.y), "=f"(b.z), "=f"(b.w) : "l"(p));
}
#if DW_NODE_Q16
struct NodeRegs { uint4 a, b, c, rf; };   // a = lo.x | lo.y, b = lo.z | hi.x, c = hi.y | hi.z (uint2 per plane), rf = references
__device__ __forceinline__ void ldg256u(const uint4* p, uint4& a, uint4& b) {
  asm volatile("ld.global.nc.v8.u32 {%0,%1,%2,%3,%4,%5,%6,%7}, [%8];"
               : "=r"(a.x), "=r"(a.y), "=r"(a.z), "=r"(a.w), "=r"(b.x), "=r"(b.y), "=r"(b.z), "=r"(b.w) : "l"(p));
}
__device__ __forceinline__ void node_load(const DwBvh& bvh, int node, NodeRegs& n) {
  const uint4* p = bvh.qnodes + 4 * (size_t)node;
  ldg256u(p, n.a, n.b); ldg256u(p + 2, n.c, n.rf);
}
__device__ __forceinline__ float q16lo(unsigned w) { return (float)(w & 0xFFFFu); }
__device__ __forceinline__ float q16hi(unsigned w) { return (float)(w >> 16); }
#else
struct NodeRegs { float4 lx, ly, lz, hx, hy, hz, rf; };
__device__ __forceinline__ void node_load(const DwBvh& bvh, int node, NodeRegs& n) {
  const float4* p = bvh.nodes + 8 * (size_t)node;
#if DW_NODE_LDG256   // three 256-bit loads for the planes, 128 bits for the references (the pad is not fetched: C2 236.4 -> 239.3, C3 222.0 -> 227.7)
  ldg256(p, n.lx, n.ly); ldg256(p + 2, n.lz, n.hx); ldg256(p + 4, n.hy, n.hz); n.rf = __ldg(p + 6);
#else
  n.lx = __ldg(p); n.ly = __ldg(p + 1); n.lz = __ldg(p + 2); n.hx = __ldg(p + 3); n.hy = __ldg(p + 4); n.hz = __ldg(p + 5); n.rf = __ldg(p + 6);
#endif
}
#endif
__device__ __forceinline__ void node_process(const DwBvh& bvh, const Ray& r, TraceState& s, const NodeRegs& n, int* sstack, int sstride, int* lstack) {
  float n0, n1, n2, n3;
#if DW_NODE_Q16
  const int r0 = (int)n.rf.x, r1 = (int)n.rf.y, r2 = (int)n.rf.z, r3 = (int)n.rf.w;
  const bool h0 = slab(r, s.best_t, bvh.eps_len, q16lo(n.a.x), q16lo(n.a.z), q16lo(n.b.x), q16lo(n.b.z), q16lo(n.c.x), q16lo(n.c.z), n0) && (r0 != DW_REF_NONE);
  const bool h1 = slab(r, s.best_t, bvh.eps_len, q16hi(n.a.x), q16hi(n.a.z), q16hi(n.b.x), q16hi(n.b.z), q16hi(n.c.x), q16hi(n.c.z), n1) && (r1 != DW_REF_NONE);
  const bool h2 = slab(r, s.best_t, bvh.eps_len, q16lo(n.a.y), q16lo(n.a.w), q16lo(n.b.y), q16lo(n.b.w), q16lo(n.c.y), q16lo(n.c.w), n2) && (r2 != DW_REF_NONE);
  const bool h3 = slab(r, s.best_t, bvh.eps_len, q16hi(n.a.y), q16hi(n.a.w), q16hi(n.b.y), q16hi(n.b.w), q16hi(n.c.y), q16hi(n.c.w), n3) && (r3 != DW_REF_NONE);
#else
  const int r0 = __float_as_int(n.rf.x), r1 = __float_as_int(n.rf.y), r2 = __float_as_int(n.rf.z), r3 = __float_as_int(n.rf.w);
  const bool h0 = slab(r, s.best_t, bvh.eps_len, n.lx.x, n.ly.x, n.lz.x, n.hx.x, n.hy.x, n.hz.x, n0) && (r0 != DW_REF_NONE);
  const bool h1 = slab(r, s.best_t, bvh.eps_len, n.lx.y, n.ly.y, n.lz.y, n.hx.y, n.hy.y, n.hz.y, n1) && (r1 != DW_REF_NONE);
  const bool h2 = slab(r, s.best_t, bvh.eps_len, n.lx.z, n.ly.z, n.lz.z, n.hx.z, n.hy.z, n.hz.z, n2) && (r2 != DW_REF_NONE);
  const bool h3 = slab(r, s.best_t, bvh.eps_len, n.lx.w, n.ly.w, n.lz.w, n.hx.w, n.hy.w, n.hz.w, n3) && (r3 != DW_REF_NONE);
#endif
  // Nearest hit child by compare-and-select on the references themselves (children of a node are distinct).  Do NOT
  // index the children by a computed position: nvcc turns that into a jump table (BRX) inside the traversal loop, and
  // on sm_100a lanes that diverge at that indirect branch were observed not to reconverge before the warp votes of
  // the schedulers (profiles/r01_pool_hang.md).
  int next = DW_REF_NONE;
  float bn = INFINITY;
  if (h0) { next = r0; bn = n0; }
  if (h1 && (next == DW_REF_NONE || n1 < bn)) { next = r1; bn = n1; }
  if (h2 && (next == DW_REF_NONE || n2 < bn)) { next = r2; bn = n2; }
  if (h3 && (next == DW_REF_NONE || n3 < bn)) { next = r3; bn = n3; }
  if (h0 && next != r0) ts_push(s, r0, sstack, sstride, lstack);
  if (h1 && next != r1) ts_push(s, r1, sstack, sstride, lstack);
  if (h2 && next != r2) ts_push(s, r2, sstack, sstride, lstack);
  if (h3 && next != r3) ts_push(s, r3, sstack, sstride, lstack);
  ts_goto(s, next, sstack, sstride, lstack);
}
#if DW_WIDE8 && !DW_NODE_Q16
// One 8-wide node: both halves are tested, the nearest hit child is visited next, the others are pushed as they lose.
__device__ __forceinline__ void step_internal(const DwBvh& bvh, const Ray& r, TraceState& s, int* sstack, int sstride, int* lstack) {
  const float4* p = bvh.nodes + 16 * (size_t)s.node;
  int next = DW_REF_NONE;
  float bn = INFINITY;
#pragma unroll
  for (int h = 0; h < 2; ++h) {
    NodeRegs n;
    n.rf = __ldg(p + 8 * h + 6);
    const int r0 = __float_as_int(n.rf.x), r1 = __float_as_int(n.rf.y), r2 = __float_as_int(n.rf.z), r3 = __float_as_int(n.rf.w);
    if (h == 1 && r0 == DW_REF_NONE) break;          // children are packed from the front: an empty first child of the second half ends it
    ldg256(p + 8 * h, n.lx, n.ly); ldg256(p + 8 * h + 2, n.lz, n.hx); ldg256(p + 8 * h + 4, n.hy, n.hz);
    float n0, n1, n2, n3;
    const bool h0 = slab(r, s.best_t, bvh.eps_len, n.lx.x, n.ly.x, n.lz.x, n.hx.x, n.hy.x, n.hz.x, n0) && (r0 != DW_REF_NONE);
    const bool h1 = slab(r, s.best_t, bvh.eps_len, n.lx.y, n.ly.y, n.lz.y, n.hx.y, n.hy.y, n.hz.y, n1) && (r1 != DW_REF_NONE);
    const bool h2 = slab(r, s.best_t, bvh.eps_len, n.lx.z, n.ly.z, n.lz.z, n.hx.z, n.hy.z, n.hz.z, n2) && (r2 != DW_REF_NONE);
    const bool h3 = slab(r, s.best_t, bvh.eps_len, n.lx.w, n.ly.w, n.lz.w, n.hx.w, n.hy.w, n.hz.w, n3) && (r3 != DW_REF_NONE);
    const int prev = next;                             // the nearest of the first half loses if this half holds a nearer one
    if (h0 && (next == DW_REF_NONE || n0 < bn)) { next = r0; bn = n0; }
    if (h1 && (next == DW_REF_NONE || n1 < bn)) { next = r1; bn = n1; }
    if (h2 && (next == DW_REF_NONE || n2 < bn)) { next = r2; bn = n2; }
    if (h3 && (next == DW_REF_NONE || n3 < bn)) { next = r3; bn = n3; }
    if (prev != DW_REF_NONE && next != prev) ts_push(s, prev, sstack, sstride, lstack);
    if (h0 && next != r0) ts_push(s, r0, sstack, sstride, lstack);
    if (h1 && next != r1) ts_push(s, r1, sstack, sstride, lstack);
    if (h2 && next != r2) ts_push(s, r2, sstack, sstride, lstack);
    if (h3 && next != r3) ts_push(s, r3, sstack, sstride, lstack);
  }
  ts_goto(s, next, sstack, sstride, lstack);
}
#else
__device__ __forceinline__ void step_internal(const DwBvh& bvh, const Ray& r, TraceState& s, int* sstack, int sstride, int* lstack) {
  NodeRegs n;
  node_load(bvh, s.node, n);
  node_process(bvh, r, s, n, sstack, sstride, lstack);
}
#endif

// One triangle of the current leaf (Moeller-Trumbore on the pre-packed record).  exclude: caller id to ignore.
// medium >= 0: only triangles whose near side (the side the ray comes from) is `medium` count (DESIGN.md
// "medium culling"); medium < 0: every triangle counts (the definition S1).  Ties -> lowest caller id.
struct TriRegs { float4 a, b, c; };
// out of line: one triangle test in ten thousand asks for it
__device__ __noinline__ float edge_slack(V3 tv, V3 pv, V3 qv, float idet) {
  return fminf(1e-5f, 4.0f * 1.1920929e-7f * (sqrtf(dot(tv, tv) * dot(pv, pv)) + sqrtf(dot(qv, qv))) * fabsf(idet));
}
__device__ __forceinline__ void ldg128v(const float4* p, float4& a) {   // volatile: the load stays where it is written (issued early)
  asm volatile("ld.global.nc.v4.f32 {%0,%1,%2,%3}, [%4];" : "=f"(a.x), "=f"(a.y), "=f"(a.z), "=f"(a.w) : "l"(p));
}
__device__ __forceinline__ void tri_load(const DwBvh& bvh, int slot, TriRegs& t) {
  const float4* p = bvh.tris + 3 * (size_t)slot;
  t.a = __ldg(p); t.b = __ldg(p + 1); t.c = __ldg(p + 2);
}
__device__ __forceinline__ void tri_load_early(const DwBvh& bvh, int slot, TriRegs& t) {
  const float4* p = bvh.tris + 3 * (size_t)slot;
  ldg128v(p, t.a); ldg128v(p + 1, t.b); ldg128v(p + 2, t.c);
}
// tback (<= 0): smallest accepted distance.  0 in a plain query.  A photon that has just left a surface (exclude >= 0) and whose
// medium is known passes -8 eps_len: its fp32 position can lie 1e-4 mm BEHIND a neighbouring facet that it would, exactly, meet
// at once (the corner between two facets of a closed shell, seen from inside, heading outwards); the medium test below keeps
// everything else out, the coplanar neighbours included, because it is made with the side the ray comes from (DESIGN.md R-seam).
__device__ __forceinline__ void tri_process(const Ray& r, TraceState& s, const TriRegs& T, int exclude, int medium, float tback,
                                            const int* sstack, int sstride, const int* lstack) {
  const float4 a = T.a, b = T.b, c = T.c;
  V3 e1 = mk(a.w, b.x, b.y), e2 = mk(b.z, b.w, c.x);
  V3 pv = cross(r.d, e2);
  float det = dot(e1, pv);
  if (fabsf(det) >= 1e-30f) {
#if DW_TRI_RCP_APPROX
    float idet = rcp_approx(det);
#else
    float idet = 1.0f / det;
#endif
    V3 tv = mk(r.o.x - a.x, r.o.y - a.y, r.o.z - a.z);
    float u = dot(tv, pv) * idet;
    V3 qv = cross(tv, e1);
    float v = dot(r.d, qv) * idet;
    float t = dot(e2, qv) * idet;
    int id = __float_as_int(c.y);
    // inside, both edges inclusive (G5), with a slack that closes the fp32 cracks between neighbours: 2e-6 for the usual ray; for a
    // ray that comes from far away onto a small triangle the rounding of u and v themselves is larger (a 1.1 m ray on a 15 mm facet
    // missed BOTH neighbours by 3e-6 and 7e-6: profiles/r02_leaks.md), so a near miss is judged again against 4 units of the
    // rounding error of the two dot products, eps (|tv| |pv| + |qv|) / |det|, at most 1e-5 (a wider band makes the owner of a point
    // between coplanar slivers a matter of rounding: first-hit ids).
    const float inside = fminf(fminf(u, v), 1.0f - (u + v));
    bool in = inside >= -kEdgeSlack;
    if (DW_EDGE_REFINE && !in && inside > -1e-5f) in = inside >= -edge_slack(tv, pv, qv, idet);
    if (in && t > tback && id != exclude && t <= fmaf(1e-6f, fabsf(t), s.best_t)) {   // a candidate: the rare part of the test
      bool ok = t > 0.f;
      if (medium >= 0) {
        const uint32_t cw = __float_as_uint(c.z);
        const int near_side = (det > 0.f) ? (int)((cw >> 8) & 0xFF) : (int)(cw & 0xFF);   // det > 0: the ray comes from the outer side
        ok = near_side == medium;
      }
      if (ok) {
        const bool thru = inside < 0.f;                      // the point lies outside this triangle by rounding, or by the slack
        bool closer = t < s.best_t || (t == s.best_t && id < (s.best_id & ~kThruSlack));
        // two neighbours met at the same distance up to rounding: the one that holds the point wins over the one that nearly
        // does (with exact arithmetic only the former is hit at all; S1)
        if (DW_EDGE_REFINE && s.best_slot >= 0 && thru != ((s.best_id & kThruSlack) != 0) && fabsf(t - s.best_t) <= 1e-6f * fabsf(t)) closer = !thru;
        if (closer) { s.best_t = t; s.best_slot = s.tri_cur; s.best_id = thru ? (id | kThruSlack) : id; }
      }
    }
  }
  if (++s.tri_cur == s.tri_end) ts_goto(s, DW_REF_NONE, sstack, sstride, lstack);
}
__device__ __forceinline__ void step_triangle(const DwBvh& bvh, const Ray& r, TraceState& s, int exclude, int medium,
                                              const int* sstack, int sstride, const int* lstack) {
  TriRegs T;
  tri_load(bvh, s.tri_cur, T);
  tri_process(r, s, T, exclude, medium, (DW_SEAM_BACK && exclude >= 0 && medium >= 0) ? -8.0f * bvh.eps_len : 0.f, sstack, sstride, lstack);
}

__global__ void __launch_bounds__(128) first_hit_kernel(DwBvh bvh, int64_t n, const float* __restrict__ ox,
                                                        const float* __restrict__ oy, const float* __restrict__ oz,
                                                        const float* __restrict__ dx, const float* __restrict__ dy,
                                                        const float* __restrict__ dz, const int32_t* __restrict__ exclude,
                                                        int32_t* __restrict__ tri, float* __restrict__ dist) {
  extern __shared__ int s_stack[];
  int lstack[kStackLocal];
  int64_t i = blockIdx.x * (int64_t)blockDim.x + threadIdx.x;
  if (i >= n) return;
  Ray r;
  ray_setup(r, mk(ox[i], oy[i], oz[i]), mk(dx[i], dy[i], dz[i]), bvh);
  TraceState s;
  ts_begin(s, INFINITY);
  const int ex = exclude ? exclude[i] : -1;
  int* my = s_stack + threadIdx.x;
  while (s.node != kDone) {
    if (s.node >= 0) step_internal(bvh, r, s, my, blockDim.x, lstack);
    else step_triangle(bvh, r, s, ex, -1, my, blockDim.x, lstack);
  }
  tri[i] = s.best_slot >= 0 ? (s.best_id & ~kThruSlack) : -1;
  dist[i] = s.best_slot >= 0 ? s.best_t : INFINITY;
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
template <class Draw>   // draw(block) -> the four uniforms of Philox block `block` of this photon and step
__device__ DW_INL_PHYS bool rayleigh(V3& k, V3& e, Draw draw) {
  for (uint32_t j = 0; j < 4096u; ++j) {
    float4 r = draw(1u + j);
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
__device__ DW_INL_PHYS void lambert(V3 nh, V3& k, V3& e, float4 r) {
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
__device__ DW_INL_PHYS uint32_t fresnel(float n1, float n2, V3 nh, V3& k, V3& e, float u, bool& crossed) {
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

// ------------------------------------------------------------------------------------------------ thin-film surface (f2)
// include/darwinopt.h "dw_set_films" (Table 8): single-film Airy summation in fp32 complex arithmetic.  Out of line on
// purpose: it is cold code, and the propagation kernels are sensitive to their instruction footprint.
struct Cf { float re, im; };
__device__ __forceinline__ Cf cf(float a, float b) { Cf z; z.re = a; z.im = b; return z; }
__device__ __forceinline__ Cf operator+(Cf a, Cf b) { return cf(a.re + b.re, a.im + b.im); }
__device__ __forceinline__ Cf operator-(Cf a, Cf b) { return cf(a.re - b.re, a.im - b.im); }
__device__ __forceinline__ Cf operator*(Cf a, Cf b) { return cf(fmaf(a.re, b.re, -a.im * b.im), fmaf(a.re, b.im, a.im * b.re)); }
__device__ __forceinline__ Cf operator*(float s, Cf a) { return cf(s * a.re, s * a.im); }
__device__ __forceinline__ Cf operator/(Cf a, Cf b) {
  float d = 1.0f / fmaf(b.re, b.re, b.im * b.im);
  return cf(fmaf(a.re, b.re, a.im * b.im) * d, fmaf(a.im, b.re, -a.re * b.im) * d);
}
__device__ __forceinline__ float cabs2(Cf a) { return fmaf(a.re, a.re, a.im * a.im); }
__device__ __forceinline__ Cf csqrtf_(Cf a) {               // principal square root
  float m = sqrtf(cabs2(a));
  float re = sqrtf(fmaxf(0.f, 0.5f * (m + a.re))), im = sqrtf(fmaxf(0.f, 0.5f * (m - a.re)));
  return cf(re, a.im < 0.f ? -im : im);
}
// Returns 0 reflected, 1 transmitted (crossed into the other medium), 2 absorbed in the film.  nh faces the photon.
// The film event inline in the film-enabled instantiation (which keeps one block fewer per SM and 96 registers): C2 with silicon-film
// cathodes 41.1 against 43.7 ms per 4e6 photons with the call; with films set and none switched on 21.2 either way (18.8 in the
// film-free instantiation).  Six blocks at 80 registers lose both ways (inline 47.3, call 46.6): profiles/r02_experiments.md 5i.
#ifndef DW_FILM_INLINE
#define DW_FILM_INLINE 1
#endif
#if DW_FILM_INLINE
#define DW_FILM_ATTR __forceinline__
#else
#define DW_FILM_ATTR __noinline__
#endif
#ifndef DW_FILM_BLOCKS_LESS
#define DW_FILM_BLOCKS_LESS 1
#endif
__device__ DW_FILM_ATTR int film_event(float n1, float nf, float kf, float d_nm, float n3, float lambda, V3 nh, V3& k, V3& e, float u) {
  const float ci = -dot(k, nh);
  const V3 sv = cross(k, nh);
  const float si2 = dot(sv, sv), si = sqrtf(si2);
  V3 s; float Es, Ep;
  if (si < 1e-5f) { s = e; Es = 1.f; Ep = 0.f; }             // normal incidence must never abort
  else { s = (1.0f / si) * sv; V3 p = cross(s, k); Es = dot(e, s); Ep = dot(e, p); }
  const Cf n2 = cf(nf, kf);
  const Cf q = cf(n1 * si, 0.f) / n2;
  Cf c2 = csqrtf_(cf(1.f, 0.f) - q * q);
  Cf n2c2 = n2 * c2;
  if (n2c2.im < 0.f || (n2c2.im == 0.f && n2c2.re < 0.f)) { c2 = cf(-c2.re, -c2.im); n2c2 = cf(-n2c2.re, -n2c2.im); }
  const float s3 = n1 * si / n3;
  const bool evan = s3 >= 1.0f;
  const Cf c3 = evan ? cf(0.f, sqrtf(s3 * s3 - 1.0f)) : cf(sqrtf(1.0f - s3 * s3), 0.f);
  // E = exp(i phi n2 c2), phi = 2 pi d / lambda
  const float phi = 6.283185307179586f * d_nm / lambda;
  float sn, cs;
  sincosf(phi * n2c2.re, &sn, &cs);
  const float mag = expf(-phi * n2c2.im);
  const Cf E = cf(mag * cs, mag * sn), E2 = E * E;
  const Cf a1 = cf(n1 * ci, 0.f), a3 = n3 * c3;             // n cos(theta) of media 1 and 3
  const Cf rs12 = (a1 - n2c2) / (a1 + n2c2), rs23 = (n2c2 - a3) / (n2c2 + a3);
  const Cf ts12 = (2.0f * a1) / (a1 + n2c2), ts23 = (2.0f * n2c2) / (n2c2 + a3);
  const Cf b1 = ci * n2, b2 = n1 * c2, b3 = n3 * c2, b4 = n2 * c3;
  const Cf rp12 = (b1 - b2) / (b1 + b2), rp23 = (b3 - b4) / (b3 + b4);
  const Cf tp12 = (2.0f * a1) / (b1 + b2), tp23 = (2.0f * n2c2) / (b3 + b4);
  const Cf one = cf(1.f, 0.f);
  const Cf ds = one + rs12 * rs23 * E2, dp = one + rp12 * rp23 * E2;
  const Cf rs = (rs12 + rs23 * E2) / ds, rp = (rp12 + rp23 * E2) / dp;
  const Cf ts = (ts12 * ts23 * E) / ds, tp = (tp12 * tp23 * E) / dp;
  const float flux = evan ? 0.f : n3 * c3.re / (n1 * ci);
  const float Rs = cabs2(rs), Rp = cabs2(rp), Ts = cabs2(ts) * flux, Tp = cabs2(tp) * flux;
  const float R = Es * Es * Rs + Ep * Ep * Rp, T = Es * Es * Ts + Ep * Ep * Tp;
  if (u < R) {
    V3 kr = unit(fma3(2.0f * ci, nh, k));
    e = unit(fma3(sqrtf(Rs) * Es, s, (sqrtf(Rp) * Ep) * cross(s, kr)));   // magnitudes kept, phases ignored (G9)
    k = kr;
    return 0;
  }
  if (u < R + T) {
    const float eta = n1 / n3, ct = sqrtf(fmaxf(0.f, 1.0f - eta * eta * si2));
    V3 kt = unit(fma3(eta, k, (eta * ci - ct) * nh));
    e = unit(fma3(sqrtf(cabs2(ts)) * Es, s, (sqrtf(cabs2(tp)) * Ep) * cross(s, kt)));
    k = kt;
    return 1;
  }
  return 2;
}

// ------------------------------------------------------------------------------------------------ empty-space look-up
// every free cell of the grid carries one box of free cells that contains it.  A segment that lies in
// such a box touches no triangle.  A segment that leaves the box of its origin's cell is followed into the box of the cell it
// enters (DW_SKIP_HOPS times): the point just behind the exit face, 8 eps_len further along the ray, starts the next test.
// That piece stays within 8 eps_len of a free cell; occupied cells are grown by 32 eps_len, of which the edge slack of the
// triangle test takes at most 15 (dw_bvh.cu grid_build), so nothing can lie on it.
#ifndef DW_SKIP_HOPS
#define DW_SKIP_HOPS 0
#endif
__device__ __forceinline__ bool free_box_of(const DwBvh& B, V3 p, V3& blo, V3& bhi) {
  const float fx = (p.x - B.grid_lo.x) * B.grid_inv_cs.x, fy = (p.y - B.grid_lo.y) * B.grid_inv_cs.y, fz = (p.z - B.grid_lo.z) * B.grid_inv_cs.z;
  const int G = B.grid_n;
  const int cx = (int)floorf(fx), cy = (int)floorf(fy), cz = (int)floorf(fz);
  if (!(cx >= 0 && cy >= 0 && cz >= 0 && cx < G && cy < G && cz < G)) return false;
  const uint2 cb = __ldg(&B.cells[(cz * G + cy) * G + cx]);
  if (!(cb.y >> 16)) return false;
  blo = mk(fmaf((float)(cb.x & 0xFF), B.grid_cs.x, B.grid_lo.x), fmaf((float)((cb.x >> 16) & 0xFF), B.grid_cs.y, B.grid_lo.y),
           fmaf((float)(cb.y & 0xFF), B.grid_cs.z, B.grid_lo.z));
  bhi = mk(fmaf((float)(((cb.x >> 8) & 0xFF) + 1), B.grid_cs.x, B.grid_lo.x), fmaf((float)(((cb.x >> 24) & 0xFF) + 1), B.grid_cs.y, B.grid_lo.y),
           fmaf((float)(((cb.y >> 8) & 0xFF) + 1), B.grid_cs.z, B.grid_lo.z));
  return p.x >= blo.x && p.x <= bhi.x && p.y >= blo.y && p.y <= bhi.y && p.z >= blo.z && p.z <= bhi.z;
}
__device__ __forceinline__ bool segment_is_free(const DwBvh& B, V3 x, V3 k, float tmax) {
  const V3 p1 = fma3(tmax, k, x);
  V3 a = x;
#pragma unroll 1
  for (int hop = 0;; ++hop) {
    V3 blo, bhi;
    if (!free_box_of(B, a, blo, bhi)) return false;
    if (p1.x >= blo.x && p1.x <= bhi.x && p1.y >= blo.y && p1.y <= bhi.y && p1.z >= blo.z && p1.z <= bhi.z) return true;
    if (hop == DW_SKIP_HOPS) return false;
    // leave the box through the face the ray meets first
    const float tx = k.x > 0.f ? (bhi.x - a.x) / k.x : (k.x < 0.f ? (blo.x - a.x) / k.x : INFINITY);
    const float ty = k.y > 0.f ? (bhi.y - a.y) / k.y : (k.y < 0.f ? (blo.y - a.y) / k.y : INFINITY);
    const float tz = k.z > 0.f ? (bhi.z - a.z) / k.z : (k.z < 0.f ? (blo.z - a.z) / k.z : INFINITY);
    const float te = fminf(fminf(tx, ty), tz);
    if (!(te >= 0.f) || !(te < INFINITY)) return false;
    a = fma3(te + 8.0f * B.eps_len, k, a);
  }
}

// L2 eviction priorities for the photon state (measured, off): a result word is stored when its photon ends, and the other seven
// photons of its 32-byte sector end up to milliseconds later; the launch moves 1.18 GB through HBM where the state is 0.76 GB.
// DW_OUT_HINT 1 / 2 / 3: result stores with L2::evict_last / .cg / .wt; DW_IN_HINT 1 / 2 / 3: input loads with L2::evict_first /
// .cs / L2::evict_last.  None lowers the traffic (profiles/r02_experiments.md section 5d): evict_last stores 1.179 GB and 0.4 ms
// slower, evict_first loads 2.74 GB (the sectors of a warp's id chunk are re-read between refills), evict_last loads 1.247 GB.
#ifndef DW_OUT_HINT
#define DW_OUT_HINT 0
#endif
#ifndef DW_IN_HINT
#define DW_IN_HINT 0
#endif
template <class T> __device__ __forceinline__ void st_out(T* p, T v) {
  static_assert(sizeof(T) == 4, "result words are 32 bits");
#if DW_OUT_HINT == 1
  unsigned long long pol;
  asm volatile("createpolicy.fractional.L2::evict_last.b64 %0, 1.0;" : "=l"(pol));
  unsigned bits;
  memcpy(&bits, &v, 4);
  asm volatile("st.global.L2::cache_hint.b32 [%0], %1, %2;" ::"l"(p), "r"(bits), "l"(pol) : "memory");
#elif DW_OUT_HINT == 2
  __stcg(p, v);
#elif DW_OUT_HINT == 3
  __stwt(p, v);
#else
  *p = v;
#endif
}
__device__ __forceinline__ float ld_in(const float* p) {
#if DW_IN_HINT == 1
  unsigned long long pol;
  asm volatile("createpolicy.fractional.L2::evict_first.b64 %0, 1.0;" : "=l"(pol));
  float v;
  asm volatile("ld.global.L2::cache_hint.f32 %0, [%1], %2;" : "=f"(v) : "l"(p), "l"(pol));
  return v;
#elif DW_IN_HINT == 2
  return __ldcs(p);
#elif DW_IN_HINT == 3
  unsigned long long pol;
  asm volatile("createpolicy.fractional.L2::evict_last.b64 %0, 1.0;" : "=l"(pol));
  float v;
  asm volatile("ld.global.L2::cache_hint.f32 %0, [%1], %2;" : "=f"(v) : "l"(p), "l"(pol));
  return v;
#else
  return *p;
#endif
}

// ------------------------------------------------------------------------------------------------ propagation
struct PropArgs {
  uint32_t keys[20];                // Philox round keys of `seed` (k0 + r W0, k1 + r W1), filled by the host: constant-bank operands
  DwBvh bvh;
  DwTables tab;
  dw_photons in;
  dw_results out;
  dw_hists hist;
  uint64_t seed;
  int32_t max_steps;
  uint32_t flags;
  int32_t th_phys, th_leaf;         // phase-scheduling thresholds (lanes)
  unsigned long long* queue_head;   // device counter, zeroed before launch
  unsigned long long* counters;     // kCount instantiation only: [kCounters] diagnostic counters, accumulated
};

// Philox4x32-10 with the round keys read from the kernel parameters (A.keys): same values as draw4(A.seed, ...).
#ifndef DW_PHILOX_KEYS
#define DW_PHILOX_KEYS 2
#endif
#ifndef DW_PHILOX_UNROLL
#define DW_PHILOX_UNROLL 10
#endif
constexpr int kPhiloxUnroll = DW_PHILOX_UNROLL;   // rounds per loop iteration of the inlined generator (10: no loop)
__device__ __forceinline__ float4 draw4_keys(const PropArgs& A, uint64_t pid, uint32_t step, uint32_t block) {
  uint4 c = make_uint4((uint32_t)pid, (uint32_t)(pid >> 32), step, block);
#pragma unroll(kPhiloxUnroll)
  for (int r = 0; r < 10; ++r) {
    uint32_t hi0 = __umulhi(0xD2511F53u, c.x), lo0 = 0xD2511F53u * c.x;
    uint32_t hi1 = __umulhi(0xCD9E8D57u, c.z), lo1 = 0xCD9E8D57u * c.z;
    c = make_uint4(hi1 ^ c.y ^ A.keys[2 * r], lo1, hi0 ^ c.w ^ A.keys[2 * r + 1], lo0);
  }
  return make_float4(u01(c.x), u01(c.y), u01(c.z), u01(c.w));
}

constexpr int kChunk = 8;   // photons claimed per lane per queue transaction (x32 per warp)

// Lane states of the persistent loop.  A warp repeatedly picks ONE of three phases and runs it for the lanes
// that are in it:
//   I  internal-node step   for lanes with ts.node >= 0
//   L  triangle step        for lanes with ts.node == kInLeaf
//   P  physics              for lanes whose query is finished (or that hold no photon: refill first)
// so that the expensive code runs with many lanes enabled although the traversals of the 32 rays of a warp
// have very different lengths (short bounded scatter segments next to long surface-to-surface rays).
enum : int { LANE_IDLE = 0, LANE_PHYS = 1, LANE_TRACE = 2 };

// kFilm: thin-film surfaces are compiled in.  Two instantiations, chosen at launch by whether dw_set_films was called: merely
// containing the (never executed) film call costs the film-free workload 21 % (C2 157 vs 199 M photons/s: spills at the call site).
template <bool kFilm>
__global__ void __launch_bounds__(128, 6) propagate_kernel(const __grid_constant__ PropArgs A) {
  extern __shared__ int s_stack[];
  __shared__ unsigned int s_fate[8];
  __shared__ unsigned long long s_steps;
  if (threadIdx.x < 8) s_fate[threadIdx.x] = 0;
  if (threadIdx.x == 0) s_steps = 0ull;
  __syncthreads();
  int* my_stack = s_stack + threadIdx.x;
  const int sstride = blockDim.x;
  int lstack[kStackLocal];
  const int lane = threadIdx.x & 31;
  const int64_t n = A.in.n;
  const bool literal = (A.flags & DW_PROP_UNBOUNDED_QUERY) != 0;

  int64_t w_next = 0, w_end = 0;     // warp-private range of photon indices; w_end < 0: queue exhausted
  int lstate = LANE_IDLE;
  bool fresh = false;                // LANE_PHYS without a finished query (photon just loaded)
  // photon state
  int64_t pi = 0;
  Ray ray;                           // ray.o = position x, ray.d = direction k
  ray.o = mk(0, 0, 0); ray.d = mk(0, 0, 1); ray.inv = mk(0, 0, 0); ray.oi = mk(0, 0, 0);
  V3 e = mk(1, 0, 0);
  float lambda = 0.f, t = 0.f;
  int medium = -1, last_tri = -1;
  uint32_t step = 0, hist = 0;
  // carried from the set-up of a query to its evaluation
  float dbulk = INFINITY, n1 = 1.f;
  bool absorb_first = false;
  TraceState ts;
  ts_begin(ts, 0.f);
  ts.node = kDone;

  for (;;) {
    const bool exhausted = w_end < 0;
    const bool tracing = lstate == LANE_TRACE;
    const int nI = __popc(__ballot_sync(0xffffffffu, tracing && ts.node >= 0));
    const int nL = __popc(__ballot_sync(0xffffffffu, tracing && ts.node == kInLeaf));
    const int nP = __popc(__ballot_sync(0xffffffffu, lstate == LANE_PHYS || (lstate == LANE_IDLE && !exhausted)));
    if (nI + nL + nP == 0) break;

    if (nI + nL > 0 && nP < A.th_phys) {
      // ------------------------------------------------------------ a4: one traversal step (phase I or L)
      if (nI > 0 && nL < A.th_leaf) {
        if (tracing && ts.node >= 0) step_internal(A.bvh, ray, ts, my_stack, sstride, lstack);
      } else {
        if (tracing && ts.node == kInLeaf)
          step_triangle(A.bvh, ray, ts, last_tri, (literal && last_tri < 0) ? -1 : medium, my_stack, sstride, lstack);
      }
      if (tracing && ts.node == kDone) { lstate = LANE_PHYS; fresh = false; }
      continue;
    }

    // -------------------------------------------------------------- phase P
    // a2: refill lanes that hold no photon from the warp's private id range
    unsigned idle = __ballot_sync(0xffffffffu, lstate == LANE_IDLE);
    if (idle && !exhausted) {
      int need = __popc(idle);
      if (w_next == w_end) {                              // claim a new chunk (one atomic per warp)
        unsigned long long base = 0;
        if (lane == 0) base = atomicAdd(A.queue_head, (unsigned long long)(32 * kChunk));
        base = __shfl_sync(0xffffffffu, base, 0);
        w_next = (int64_t)base;
        w_end = (int64_t)base + 32 * kChunk;
        if (w_next >= n) { w_next = 0; w_end = -1; }
        else if (w_end > n) w_end = n;
      }
      if (w_end > w_next) {
        int rank = __popc(idle & ((1u << lane) - 1u));
        int avail = (int)min((int64_t)need, w_end - w_next);
        if (lstate == LANE_IDLE && rank < avail) {
          pi = w_next + rank;
          ray.o = mk(A.in.px[pi], A.in.py[pi], A.in.pz[pi]);
          ray.d = mk(A.in.kx[pi], A.in.ky[pi], A.in.kz[pi]);
          e = mk(A.in.ex[pi], A.in.ey[pi], A.in.ez[pi]);
          lambda = A.in.wavelength[pi];
          t = A.in.t0[pi];
          medium = -1; last_tri = -1; step = 0; hist = 0;
          lstate = LANE_PHYS; fresh = true;
        }
        w_next += avail;
      }
    }

    uint32_t fate = 0xFFu;           // 0xFF = still running
    int channel = -1;
    if (lstate == LANE_PHYS) {
      const uint64_t pid = A.in.photon_id_base + (uint64_t)pi;
      V3 x = ray.o, k = ray.d;
      if (!fresh) {
        // ---------------------------------------------------------- evaluate the finished query: S2..S9
        float4 r0 = draw4(A.seed, pid, step, 0u);                     // (u_a, u_s, u_surface, u_fresnel)
        const bool bounded = (!literal) && (medium >= 0);
        const bool have_hit = ts.best_slot >= 0;
        float4 tc = make_float4(0, 0, 0, 0), ta = tc, tb = tc;
        int m1 = medium, m2 = medium;
        V3 ng = mk(0, 0, 1);
        bool toward_outer = false;
        if (have_hit) {                                               // S2 sides
          const float4* p = A.bvh.tris + 3 * (size_t)ts.best_slot;
          ta = __ldg(p); tb = __ldg(p + 1); tc = __ldg(p + 2);
          ng = unit(cross(mk(ta.w, tb.x, tb.y), mk(tb.z, tb.w, tc.x)));
          uint32_t cw = __float_as_uint(tc.z);
          toward_outer = dot(k, ng) > 0.f;
          int mi = (int)(cw & 0xFF), mo = (int)((cw >> 8) & 0xFF);
          m1 = toward_outer ? mi : mo;
          m2 = toward_outer ? mo : mi;
        }
        if (!bounded) {
          if (!have_hit) {
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
          const bool surface_event = have_hit && (bounded ? true : !(dbulk < ts.best_t));
          if (!surface_event) {
            if (!(dbulk < INFINITY)) {
              fate = DW_FATE_ESCAPED;                                 // bounded query, no bulk process, nothing hit
            } else {
              x = fma3(dbulk, k, x);
              t = fmaf(dbulk * n1, kInvC, t);
              if (absorb_first) {
                fate = DW_FATE_BULK_ABSORBED;                         // S4 first branch
              } else {                                                // S4 second branch + S6
                if (!rayleigh(k, e, [&](uint32_t b) { return draw4(A.seed, pid, step, b); })) fate = DW_FATE_NAN_ABORT;
                hist |= DW_H_RAYLEIGH;
                last_tri = -1;
              }
            }
          } else {                                                    // S4 third branch, S5
            x = fma3(ts.best_t, k, x);
            t = fmaf(ts.best_t * n1, kInvC, t);
            last_tri = ts.best_id & ~kThruSlack;
            if (medium != m1) hist |= DW_H_MEDIUM_MISMATCH;
            V3 nh = toward_outer ? mk(-ng.x, -ng.y, -ng.z) : ng;
            uint32_t cw = __float_as_uint(tc.z);
            int sf = (int)((cw >> 16) & 0xFF);
            bool is_film = false;
            if constexpr (kFilm) is_film = sf != 0xFF && __ldg(&A.tab.film_on[sf]) != 0;
            if (is_film) {                                            // thin-film surface (second mode)
              const size_t ss = (size_t)A.tab.n_surf * A.tab.nl_surf;
              const float n3 = table_at(A.tab.mat, m2, A.tab.nl_mat, A.tab.mat_l0, A.tab.mat_inv_dl, lambda);
              const float fnf = table_at(A.tab.film, sf, A.tab.nl_surf, A.tab.surf_l0, A.tab.surf_inv_dl, lambda);
              const float fkf = table_at(A.tab.film + ss, sf, A.tab.nl_surf, A.tab.surf_l0, A.tab.surf_inv_dl, lambda);
              const float fd = table_at(A.tab.film + 2 * ss, sf, A.tab.nl_surf, A.tab.surf_l0, A.tab.surf_inv_dl, lambda);
              int oc = 2;
              if constexpr (kFilm) oc = film_event(n1, fnf, fkf, fd, n3, lambda, nh, k, e, r0.w);
              hist |= DW_H_FILM;
              if (oc == 0) hist |= DW_H_REFLECT_SPECULAR;
              else if (oc == 1) { hist |= DW_H_SURFACE_TRANSMIT; medium = m2; }
              else if (r0.z < table_at(A.tab.surf, sf, A.tab.nl_surf, A.tab.surf_l0, A.tab.surf_inv_dl, lambda)) { fate = DW_FATE_DETECTED; channel = __float_as_int(tc.w); }
              else fate = DW_FATE_SURFACE_ABSORBED;
            } else if (sf != 0xFF) {                                  // S7 explicit surface
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
        }
        ++step;                                                       // S9 (every executed iteration counts, also the last: S13)
      }
      if (fate == 0xFFu) {
        // ---------------------------------------------------------- set up the query of the next iteration: S1 (+S3/S4 draws)
        if ((int32_t)step >= A.max_steps) {
          fate = DW_FATE_TRUNCATED;                                   // S10
        } else if (!(isfinite(x.x + x.y + x.z) && isfinite(k.x + k.y + k.z) && isfinite(e.x + e.y + e.z) && isfinite(t))) {
          fate = DW_FATE_NAN_ABORT;                                   // S11
        } else {
          float tmax = INFINITY;
          if ((!literal) && medium >= 0) {                            // medium known: S3/S4 draws before the query
            float4 r0 = draw4(A.seed, pid, step, 0u);
            n1 = table_at(A.tab.mat, medium, A.tab.nl_mat, A.tab.mat_l0, A.tab.mat_inv_dl, lambda);
            float La = table_at(A.tab.mat + (size_t)A.tab.n_mat * A.tab.nl_mat, medium, A.tab.nl_mat, A.tab.mat_l0, A.tab.mat_inv_dl, lambda);
            float Ls = table_at(A.tab.mat + 2 * (size_t)A.tab.n_mat * A.tab.nl_mat, medium, A.tab.nl_mat, A.tab.mat_l0, A.tab.mat_inv_dl, lambda);
            float da = -La * logf(r0.x), ds = -Ls * logf(r0.y);
            absorb_first = da < ds;
            dbulk = fminf(da, ds);
            tmax = dbulk + A.bvh.eps_len;
          }
          ray_setup(ray, x, k, A.bvh);
          ts_begin(ts, tmax);
          lstate = LANE_TRACE;
          fresh = false;
        }
      }
      ray.o = x; ray.d = k;
    }

    // ---------------------------------------------------------------- a10: outputs and reductions
    if (fate != 0xFFu) {
      if (A.out.flags) A.out.flags[pi] = fate | hist;
      if (A.out.channel) A.out.channel[pi] = channel;
      if (A.out.t) A.out.t[pi] = t;
      if (A.out.steps) A.out.steps[pi] = step;
      if (A.out.last_tri) A.out.last_tri[pi] = last_tri;
      if (A.out.x) A.out.x[pi] = ray.o.x;
      if (A.out.y) A.out.y[pi] = ray.o.y;
      if (A.out.z) A.out.z[pi] = ray.o.z;
      if (A.out.kx) { A.out.kx[pi] = ray.d.x; A.out.ky[pi] = ray.d.y; A.out.kz[pi] = ray.d.z; }
      if (A.out.ex) { A.out.ex[pi] = e.x; A.out.ey[pi] = e.y; A.out.ez[pi] = e.z; }
      atomicAdd(&s_fate[fate & 7u], 1u);
      atomicAdd(&s_steps, (unsigned long long)step);
      lstate = LANE_IDLE;
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

// ------------------------------------------------------------------------------------------------ propagation, pool scheduler
// Second scheduler: every warp owns kSlots photon slots in shared memory (SoA, one
// word per field per slot).  A slot is EMPTY, waits for physics (PHYS: query finished), waits for a lane (TRACE:
// next query set up) or is being traced by a lane (BUSY).  Lanes keep only the ray and the traversal state of the
// query they run; when a query ends the lane writes (best_t, best_slot) to the slot and fetches another TRACE slot,
// so traversal does not wait for physics, and physics runs for 32 slots at a time with every lane enabled.
#ifndef DW_POOL_SLOTS
#define DW_POOL_SLOTS 64
#endif
constexpr int kSlots = DW_POOL_SLOTS;      // 33..96: lane l looks after slots l, l + 32 and l + 64 (those that exist)
static_assert(kSlots > 32 && kSlots <= 96, "pool size");
// The last two words exist only in the full layout: with flat tables and no films the wavelength is never read again and n1 is one
// table load from the medium, so the lean layout (20 words) leaves them out.  With 8 shared stack entries a lean block takes 26 kB, six of
// them fit the 164 kB shared-memory configuration instead of 196 kB, and L1 grows from ~60 to ~92 kB (profiles/r01_captures_9_to_12_c2.md).
enum : int { W_X = 0, W_Y, W_Z, W_KX, W_KY, W_KZ, W_EX, W_EY, W_EZ, W_T, W_MEDIUM, W_LAST, W_STEP, W_HIST, W_PI,
             W_DBULK, W_US, W_UF, W_BEST_T, W_BEST_SLOT, kWordsLean, W_LAMBDA = kWordsLean, W_N1, kWordsFull };
enum : int { S_EMPTY = 0, S_PHYS = 1, S_TRACE = 2, S_BUSY = 3 };
constexpr uint32_t kAbsorbFirstBit = 0x80000000u;                 // kept in the W_HIST word
// per-warp layout in ints: pool[words][kSlots], status[kSlots], queue[kSlots] (rank -> slot scratch), stack[kStackShared][32]
constexpr int warp_st(bool lean) { return (lean ? kWordsLean : kWordsFull) * kSlots; }
constexpr int warp_q(bool lean) { return warp_st(lean) + kSlots; }
constexpr int warp_stack(bool lean) { return warp_q(lean) + kSlots; }
constexpr int warp_ints(bool lean) { return warp_stack(lean) + kStackShared * 32; }

// 6 resident blocks (24 warps) per SM: 80 registers, no spills; measured on C2 against 4 blocks (118 registers): 134 vs 117 M photons/s.
#ifndef DW_POOL_MIN_BLOCKS
#define DW_POOL_MIN_BLOCKS 6
#endif
#ifndef DW_NODE_REPS
#define DW_NODE_REPS 2
#endif
#ifndef DW_TRI_REPS
#define DW_TRI_REPS 2
#endif
// Slots that must be ready for a physics phase before tracing lanes that find nothing queued leave the traversal loop for it.  The
// pool of 64 slots never holds less than 32 ready slots when 8 lanes are idle, so 32 means "whenever th_phys lanes starve"; 16 lets
// a warp in its tail do the same.  C2 42.46 -> 42.14 ms, C3 44.76 -> 44.46 (12 / 16 / 20 within 0.1 ms; profiles/r02_experiments.md 5e).
#ifndef DW_TH_READY
#define DW_TH_READY 16
#endif
// Ready slots from which a physics phase runs whatever the lanes are doing (a phase takes at most 32).  Phases with fewer slots cost
// the same instructions: 28 / 24 / 20 / 16 measured 42.9 / 44.5 / 46.7 / 49.0 against 42.4 ms.
#ifndef DW_REFILL_MIN
#define DW_REFILL_MIN 0
#endif
#ifndef DW_TH_PHYS_FULL
#define DW_TH_PHYS_FULL 32
#endif
#ifndef DW_NODE_REPS_MIN
#define DW_NODE_REPS_MIN 16
#endif
#ifndef DW_TRI_PAIR
#define DW_TRI_PAIR 0   // measured: 42.4 against 41.6 ms on C2 (profiles/r02_experiments.md)
#endif

// The film-enabled instantiation gets one block fewer per SM: at 80 registers it spills 106 bytes around the film call.
// kFlat: all tables have one wavelength node (the BASELINE.json configs): a look-up is one load, no call.
// The Rayleigh loop S6 runs at most DW_RAYL_REQUEUE iterations inside a physics phase; a slot that is still rejected then goes back
// to the list of the phase with its iteration number and continues in the next one, with a phase full of slots.  (The whole loop
// inside the phase ran its later iterations for the few lanes still rejected: 9 of 32 lanes on average over the loop; one iteration
// per phase costs more in slot traffic than it saves: profiles/r02_experiments.md.)  Draws are keyed by (photon, step, block 1 + j):
// same results.  0: the loop of the first build.
// DW_RAYL_COOP 1: the loop S6 for all lanes of a phase together, every lane of the warp drawing one candidate for one of the
// scattering photons (up to four candidates per photon and round; results bit-identical).  Measured: 18.5 instead of 15.6 lanes per
// instruction, the same number of instructions, 1.4 kB more code -> 0.95 instead of 0.33 stall cycles per instruction waiting for
// instructions, 44.7 against 42.1 ms (profiles/r02_experiments.md section 5h).  Off.
#ifndef DW_RAYL_COOP
#define DW_RAYL_COOP 0
#endif
#ifndef DW_RAYL_REQUEUE
#define DW_RAYL_REQUEUE 0
#endif
constexpr int kRaylPending = -2;           // W_BEST_SLOT <= kRaylPending: iteration kRaylPending - W_BEST_SLOT of S6 is due
// diagnostic counters of the kCount instantiation (dw_propagate_counters)
enum : int { C_NODE = 0, C_TRI, C_TRACED, C_SKIPPED, C_PHASES, C_LANES_PHYS, C_LANES_RAYL, C_LANES_SETUP, C_LANES_FRESH, C_ITER_NODE, C_LANES_NODE,
             C_ITER_LEAF, C_LANES_LEAF, C_FETCH, C_LANES_FETCH, C_RAYL_ITER,
             C_Q_FRESH, C_N_FRESH, C_Q_SURF, C_N_SURF, C_H_SURF, C_Q_BULK, C_N_BULK, C_H_BULK, kCounters = 24 };

template <bool kFilm, bool kFlat, bool kCount>
__global__ void __launch_bounds__(128, kFilm ? DW_POOL_MIN_BLOCKS - DW_FILM_BLOCKS_LESS : DW_POOL_MIN_BLOCKS) propagate_pool_kernel(const __grid_constant__ PropArgs A) {
  extern __shared__ int s_dyn[];
  __shared__ unsigned long long s_cnt[kCount ? kCounters : 1];
  if constexpr (kCount) { if (threadIdx.x < kCounters) s_cnt[threadIdx.x] = 0ull; }
#define CNT(i, v) do { if constexpr (kCount) { if ((threadIdx.x & 31) == 0) atomicAdd(&s_cnt[i], (unsigned long long)(v)); } } while (0)
  auto TAB = [](const float* __restrict__ tab, int row, int nl, float l0, float inv_dl, float lam) -> float {
    if constexpr (kFlat) return __ldg(tab + row);
    else return table_at(tab, row, nl, l0, inv_dl, lam);
  };
  // Philox at the two hot sites (block 0 of the next query, the Rayleigh loop) and at the cold ones (first step, Lambert)
  auto DRAW_HOT = [&](uint64_t pid_, uint32_t step_, uint32_t block_) -> float4 {
    if constexpr (DW_PHILOX_KEYS >= 1) return draw4_keys(A, pid_, step_, block_);
    else return draw4(A.seed, pid_, step_, block_);
  };
  auto DRAW_COLD = [&](uint64_t pid_, uint32_t step_, uint32_t block_) -> float4 {
    if constexpr (DW_PHILOX_KEYS >= 2) return draw4_keys(A, pid_, step_, block_);
    else return draw4(A.seed, pid_, step_, block_);
  };
  __shared__ unsigned int s_fate[8];
  __shared__ unsigned long long s_steps;
  if (threadIdx.x < 8) s_fate[threadIdx.x] = 0;
  if (threadIdx.x == 0) s_steps = 0ull;
  const int lane = threadIdx.x & 31;
  constexpr bool kLean = kFlat && !kFilm;
  int* const wbase = s_dyn + (threadIdx.x >> 5) * warp_ints(kLean);
  int* const pool = wbase;
  float* const poolf = reinterpret_cast<float*>(wbase);
  int* const st = wbase + warp_st(kLean);
  int* const q = wbase + warp_q(kLean);
  int* const my_stack = wbase + warp_stack(kLean) + lane;
  constexpr int sstride = 32;
  const bool has2 = lane + 32 < kSlots;            // this lane also looks after slot lane + 32
  const bool has3 = lane + 64 < kSlots;            // ... and slot lane + 64 (pools of more than 64 slots)
  st[lane] = S_EMPTY;
  if (has2) st[lane + 32] = S_EMPTY;
  if (has3) st[lane + 64] = S_EMPTY;
  __syncthreads();
  int lstack[kStackLocal];
  const unsigned lt = (1u << lane) - 1u;
  const int64_t n = A.in.n;
  const bool literal = (A.flags & DW_PROP_UNBOUNDED_QUERY) != 0;
  const int th_fetch = A.th_phys, th_leaf = A.th_leaf;
  const bool use_grid = A.bvh.cells != nullptr && !(A.flags & DW_PROP_NO_EMPTY_SKIP);

  int64_t w_next = 0, w_end = 0;     // warp-private range of photon indices
  bool exhausted = false;
  // the query this lane is running
  int my = -1;                       // slot, -1: lane idle
  Ray ray;
  ray.o = mk(0, 0, 0); ray.d = mk(0, 0, 1); ray.inv = mk(0, 0, 0); ray.oi = mk(0, 0, 0);
  int q_exclude = -1, q_medium = -1;
  TraceState ts;
  ts_begin(ts, 0.f);
  ts.node = kDone;
  [[maybe_unused]] int my_visits = 0;   // kCount: box-node visits of the running query

  for (;;) {
    // ---------------------------------------------------------------- census of the warp's slots
    const int s0 = st[lane], s1 = has2 ? st[lane + 32] : -1;
    int s2 = -1;
    if constexpr (kSlots > 64) s2 = has3 ? st[lane + 64] : -1;
    const unsigned p0 = __ballot_sync(0xffffffffu, s0 == S_PHYS), p1 = __ballot_sync(0xffffffffu, s1 == S_PHYS);
    const unsigned e0 = __ballot_sync(0xffffffffu, s0 == S_EMPTY), e1 = __ballot_sync(0xffffffffu, s1 == S_EMPTY);
    const unsigned t0 = __ballot_sync(0xffffffffu, s0 == S_TRACE), t1 = __ballot_sync(0xffffffffu, s1 == S_TRACE);
    unsigned p2 = 0, e2 = 0, t2 = 0;
    if constexpr (kSlots > 64) {
      p2 = __ballot_sync(0xffffffffu, s2 == S_PHYS); e2 = __ballot_sync(0xffffffffu, s2 == S_EMPTY); t2 = __ballot_sync(0xffffffffu, s2 == S_TRACE);
    }
    const unsigned idle = __ballot_sync(0xffffffffu, my < 0);
    const int nP = __popc(p0) + __popc(p1) + __popc(p2);
    const int nE = exhausted ? 0 : __popc(e0) + __popc(e1) + __popc(e2);
    const int nQ = __popc(t0) + __popc(t1) + __popc(t2);
    const int nB = 32 - __popc(idle);
    if (nP + nE + nQ + nB == 0) break;

    const bool do_phys = (nP + nE >= DW_TH_PHYS_FULL) || (nQ == 0 && (nB == 0 || nP + nE >= 8));
    if (do_phys) {
      // -------------------------------------------------------------- phase P: up to 32 slots, finished queries first
      const int nPc = min(nP, 32 - min(nE, DW_REFILL_MIN)); // finished queries first, but DW_REFILL_MIN lanes are kept for empty slots
      int take = min(nE, 32 - nPc);                         // empty slots to refill (a2)
      if (take > 0 && w_next == w_end) {                    // claim a new chunk of photon ids (one atomic per warp)
        unsigned long long base = 0;
        if (lane == 0) base = atomicAdd(A.queue_head, (unsigned long long)(32 * kChunk));
        base = __shfl_sync(0xffffffffu, base, 0);
        w_next = (int64_t)base;
        w_end = (int64_t)base + 32 * kChunk;
        if (w_next >= n) { w_next = w_end = 0; exhausted = true; }
        else if (w_end > n) w_end = n;
      }
      take = (int)min((int64_t)take, w_end - w_next);
      if (s0 == S_PHYS) q[__popc(p0 & lt)] = lane;
      if (s1 == S_PHYS) q[__popc(p0) + __popc(p1 & lt)] = lane + 32;
      if (s0 == S_EMPTY) q[nP + __popc(e0 & lt)] = lane;
      if (s1 == S_EMPTY) q[nP + __popc(e0) + __popc(e1 & lt)] = lane + 32;
      if constexpr (kSlots > 64) {
        if (s2 == S_PHYS) q[__popc(p0) + __popc(p1) + __popc(p2 & lt)] = lane + 64;
        if (s2 == S_EMPTY) q[nP + __popc(e0) + __popc(e1) + __popc(e2 & lt)] = lane + 64;
      }
      __syncwarp();
      int slot = -1;
      bool fresh = false;
      int64_t pi = 0;
      if (lane < nPc) slot = q[lane];
      else if (lane < nPc + take) { slot = q[nP + (lane - nPc)]; fresh = true; pi = w_next + (lane - nPc); }
      w_next += take;
      if (nPc + take == 0) continue;                        // nothing to do this round (queue just ran dry)
      CNT(C_PHASES, 1); CNT(C_LANES_PHYS, nPc); CNT(C_LANES_FRESH, take);

      V3 x = mk(0, 0, 0), k = mk(0, 0, 1), e = mk(1, 0, 0);
      float lambda = 0.f, t = 0.f, dbulk = INFINITY, n1 = 1.f, us = 0.f, uf = 0.f, best_t = INFINITY;
      int medium = -1, last_tri = -1, best_slot = -1;
      uint32_t step = 0, hist = 0;
      bool absorb_first = false;
      if (fresh) {
        x = mk(ld_in(A.in.px + pi), ld_in(A.in.py + pi), ld_in(A.in.pz + pi));
        k = mk(ld_in(A.in.kx + pi), ld_in(A.in.ky + pi), ld_in(A.in.kz + pi));
        e = mk(ld_in(A.in.ex + pi), ld_in(A.in.ey + pi), ld_in(A.in.ez + pi));
        lambda = ld_in(A.in.wavelength + pi);
        t = ld_in(A.in.t0 + pi);
      } else if (slot >= 0) {
        x = mk(poolf[W_X * kSlots + slot], poolf[W_Y * kSlots + slot], poolf[W_Z * kSlots + slot]);
        k = mk(poolf[W_KX * kSlots + slot], poolf[W_KY * kSlots + slot], poolf[W_KZ * kSlots + slot]);
        e = mk(poolf[W_EX * kSlots + slot], poolf[W_EY * kSlots + slot], poolf[W_EZ * kSlots + slot]);
        if constexpr (!kLean) lambda = poolf[W_LAMBDA * kSlots + slot];
        t = poolf[W_T * kSlots + slot];
        medium = pool[W_MEDIUM * kSlots + slot];
        last_tri = pool[W_LAST * kSlots + slot];
        step = (uint32_t)pool[W_STEP * kSlots + slot];
        hist = (uint32_t)pool[W_HIST * kSlots + slot];
        absorb_first = (hist & kAbsorbFirstBit) != 0;
        hist &= ~kAbsorbFirstBit;
        pi = (int64_t)(uint32_t)pool[W_PI * kSlots + slot];
        dbulk = poolf[W_DBULK * kSlots + slot];
        if constexpr (!kLean) n1 = poolf[W_N1 * kSlots + slot];
        us = poolf[W_US * kSlots + slot];
        uf = poolf[W_UF * kSlots + slot];
        best_t = poolf[W_BEST_T * kSlots + slot];
        best_slot = pool[W_BEST_SLOT * kSlots + slot];
        if constexpr (kLean) { if (medium >= 0) n1 = __ldg(A.tab.mat + medium); }   // the value the query set-up computed
      }
      uint32_t fate = 0xFFu;           // 0xFF = still running
      int channel = -1;
      const uint64_t pid = A.in.photon_id_base + (uint64_t)pi;
      int rj = -1;                     // iteration of the Rayleigh loop S6 that this lane runs in this phase (-1: none)
      if (DW_RAYL_REQUEUE && slot >= 0 && !fresh && best_slot <= kRaylPending) rj = kRaylPending - best_slot;
      if (slot >= 0 && !fresh && rj < 0) {
        // ---------------------------------------------------------- evaluate the finished query: S2..S9
        const bool bounded = (!literal) && (medium >= 0);
        const bool have_hit = best_slot >= 0;
        float4 tc = make_float4(0, 0, 0, 0), ta = tc, tb = tc;
        int m1 = medium, m2 = medium;
        V3 ng = mk(0, 0, 1);
        bool toward_outer = false;
        if (have_hit) {                                               // S2 sides
          const float4* p = A.bvh.tris + 3 * (size_t)best_slot;
          ta = __ldg(p); tb = __ldg(p + 1); tc = __ldg(p + 2);
          ng = unit(cross(mk(ta.w, tb.x, tb.y), mk(tb.z, tb.w, tc.x)));
          uint32_t cw = __float_as_uint(tc.z);
          toward_outer = dot(k, ng) > 0.f;
          int mi = (int)(cw & 0xFF), mo = (int)((cw >> 8) & 0xFF);
          m1 = toward_outer ? mi : mo;
          m2 = toward_outer ? mo : mi;
        }
        if (!bounded) {
          if (!have_hit) {
            fate = DW_FATE_ESCAPED;                                   // G3: ray leaves the world
          } else {
            float4 r0 = DRAW_COLD(pid, step, 0u);                 // (u_a, u_s, u_surface, u_fresnel)
            us = r0.z; uf = r0.w;
            if (medium >= 0 && medium != m1) hist |= DW_H_MEDIUM_MISMATCH;
            medium = m1;
            n1 = TAB(A.tab.mat, m1, A.tab.nl_mat, A.tab.mat_l0, A.tab.mat_inv_dl, lambda);
            float La = TAB(A.tab.mat + (size_t)A.tab.n_mat * A.tab.nl_mat, m1, A.tab.nl_mat, A.tab.mat_l0, A.tab.mat_inv_dl, lambda);
            float Ls = TAB(A.tab.mat + 2 * (size_t)A.tab.n_mat * A.tab.nl_mat, m1, A.tab.nl_mat, A.tab.mat_l0, A.tab.mat_inv_dl, lambda);
            float da = -La * logf(r0.x), ds = -Ls * logf(r0.y);
            absorb_first = da < ds;
            dbulk = fminf(da, ds);
          }
        }
        if (fate == 0xFFu) {
          const bool surface_event = have_hit && (bounded ? true : !(dbulk < best_t));
          if (!surface_event) {
            if (!(dbulk < INFINITY)) {
              fate = DW_FATE_ESCAPED;                                 // bounded query, no bulk process, nothing hit
            } else {
              x = fma3(dbulk, k, x);
              t = fmaf(dbulk * n1, kInvC, t);
              if (absorb_first) {
                fate = DW_FATE_BULK_ABSORBED;                         // S4 first branch
              } else {                                                // S4 second branch + S6
#if DW_RAYL_REQUEUE || DW_RAYL_COOP
                rj = 0;                                               // the loop runs below, for all lanes of the phase together
                --step;                                               // S9 counts the step when the loop ends
#else
                if (!rayleigh(k, e, [&](uint32_t b) { return DRAW_HOT(pid, step, b); })) fate = DW_FATE_NAN_ABORT;
#endif
                hist |= DW_H_RAYLEIGH;
                last_tri = -1;
              }
            }
          } else {                                                    // S4 third branch, S5
            x = fma3(best_t, k, x);
            t = fmaf(best_t * n1, kInvC, t);
            last_tri = __float_as_int(tc.y);
            if (medium != m1) hist |= DW_H_MEDIUM_MISMATCH;
            V3 nh = toward_outer ? mk(-ng.x, -ng.y, -ng.z) : ng;
            uint32_t cw = __float_as_uint(tc.z);
            int sf = (int)((cw >> 16) & 0xFF);
            bool is_film = false;
            if constexpr (kFilm) is_film = sf != 0xFF && __ldg(&A.tab.film_on[sf]) != 0;
            if (is_film) {                                            // thin-film surface (second mode)
              const size_t ss = (size_t)A.tab.n_surf * A.tab.nl_surf;
              const float n3 = TAB(A.tab.mat, m2, A.tab.nl_mat, A.tab.mat_l0, A.tab.mat_inv_dl, lambda);
              const float fnf = TAB(A.tab.film, sf, A.tab.nl_surf, A.tab.surf_l0, A.tab.surf_inv_dl, lambda);
              const float fkf = TAB(A.tab.film + ss, sf, A.tab.nl_surf, A.tab.surf_l0, A.tab.surf_inv_dl, lambda);
              const float fd = TAB(A.tab.film + 2 * ss, sf, A.tab.nl_surf, A.tab.surf_l0, A.tab.surf_inv_dl, lambda);
              int oc = 2;
              if constexpr (kFilm) oc = film_event(n1, fnf, fkf, fd, n3, lambda, nh, k, e, uf);
              hist |= DW_H_FILM;
              if (oc == 0) hist |= DW_H_REFLECT_SPECULAR;
              else if (oc == 1) { hist |= DW_H_SURFACE_TRANSMIT; medium = m2; }
              else if (us < TAB(A.tab.surf, sf, A.tab.nl_surf, A.tab.surf_l0, A.tab.surf_inv_dl, lambda)) { fate = DW_FATE_DETECTED; channel = __float_as_int(tc.w); }
              else fate = DW_FATE_SURFACE_ABSORBED;
            } else if (sf != 0xFF) {                                  // S7 explicit surface
              const size_t ss = (size_t)A.tab.n_surf * A.tab.nl_surf;
              float c0 = TAB(A.tab.surf, sf, A.tab.nl_surf, A.tab.surf_l0, A.tab.surf_inv_dl, lambda);
              float c1 = TAB(A.tab.surf + ss, sf, A.tab.nl_surf, A.tab.surf_l0, A.tab.surf_inv_dl, lambda);
              float c2 = TAB(A.tab.surf + 2 * ss, sf, A.tab.nl_surf, A.tab.surf_l0, A.tab.surf_inv_dl, lambda);
              float c3 = TAB(A.tab.surf + 3 * ss, sf, A.tab.nl_surf, A.tab.surf_l0, A.tab.surf_inv_dl, lambda);
              if (us < c0) { fate = DW_FATE_DETECTED; channel = __float_as_int(tc.w); }
              else if (us < c1) { lambert(nh, k, e, DRAW_COLD(pid, step, 1u)); hist |= DW_H_REFLECT_DIFFUSE; }
              else if (us < c2) {                                     // specular: no plane of incidence needed
                k = unit(fma3(-2.0f * dot(k, nh), nh, k));
                e = unit(fma3(-2.0f * dot(e, nh), nh, e));
                hist |= DW_H_REFLECT_SPECULAR;
              }
              else if (us < c3) { hist |= DW_H_SURFACE_TRANSMIT; medium = m2; }
              else fate = DW_FATE_SURFACE_ABSORBED;
            } else {                                                  // S8 Fresnel
              float n2 = TAB(A.tab.mat, m2, A.tab.nl_mat, A.tab.mat_l0, A.tab.mat_inv_dl, lambda);
              bool crossed;
              hist |= fresnel(n1, n2, nh, k, e, uf, crossed);
              if (crossed) medium = m2;
            }
          }
        }
        ++step;                                                       // S9 (every executed iteration counts, also the last: S13)
      }
#if DW_RAYL_COOP
      // S6 for all lanes of the phase together.  The rejection loop accepts two candidates in three, so run lane by lane it takes the
      // warp four iterations at nine, three, one lanes.  Here every lane of the warp draws ONE candidate for one of the nR scattering
      // photons: lane l serves the photon of rank l % nR with candidate number rj + l / nR (Philox block 1 + that number, as in the
      // loop), and a photon takes its accepted candidate of lowest number: the same direction and polarisation as the loop's.
#pragma unroll 1
      for (;;) {
        const unsigned rm = __ballot_sync(0xffffffffu, rj >= 0);
        if (!rm) break;
        const int nR = __popc(rm);
        const int rank = __popc(rm & lt);
        CNT(C_RAYL_ITER, 1); CNT(C_LANES_RAYL, nR);
        __syncwarp();
        if (rj >= 0) q[rank] = lane;
        __syncwarp();
        const int cand = (lane >= nR) + (lane >= 2 * nR) + (lane >= 3 * nR);   // lane / nR, at most four candidates per photon and round
        const int src = q[min(lane - cand * nR, nR - 1)];             // the lane whose photon this lane draws for (lanes >= 4 nR: unused)
        const uint32_t pi_r = __shfl_sync(0xffffffffu, (uint32_t)pi, src), step_r = __shfl_sync(0xffffffffu, step, src);
        const int rj_r = __shfl_sync(0xffffffffu, rj, src);
        const V3 e_r = mk(__shfl_sync(0xffffffffu, e.x, src), __shfl_sync(0xffffffffu, e.y, src), __shfl_sync(0xffffffffu, e.z, src));
        const float4 r = DRAW_HOT(A.in.photon_id_base + (uint64_t)pi_r, step_r, 1u + (uint32_t)(rj_r + cand));
        const float ct = 1.0f - 2.0f * r.x;
        const float st_ = sqrtf(fmaxf(0.f, 1.0f - ct * ct));
        float sp, cp;
        sincospif(2.0f * r.y, &sp, &cp);
        const V3 kn = mk(st_ * cp, st_ * sp, ct);
        V3 er = fma3(-dot(e_r, kn), kn, e_r);
        const float w = dot(er, er);
        er = rsqrtf(w) * er;
        const unsigned acc = __ballot_sync(0xffffffffu, r.z < w && lane < 4 * nR);
        const unsigned stride = 1u | (nR < 32 ? 1u << nR : 0u) | (2 * nR < 32 ? 1u << (2 * nR) : 0u) | (3 * nR < 32 ? 1u << (3 * nR) : 0u);
        const unsigned mine = stride << rank;                         // the lanes that drew for this lane's photon (lanes >= 32 drop out)
        const int win = __ffs(acc & mine) - 1;
        const int from = win >= 0 ? win : lane;
        const V3 kw = mk(__shfl_sync(0xffffffffu, kn.x, from), __shfl_sync(0xffffffffu, kn.y, from), __shfl_sync(0xffffffffu, kn.z, from));
        const V3 ew = mk(__shfl_sync(0xffffffffu, er.x, from), __shfl_sync(0xffffffffu, er.y, from), __shfl_sync(0xffffffffu, er.z, from));
        if (rj >= 0) {
          if (win >= 0) { k = kw; e = ew; ++step; rj = -1; }                                        // S9
          else if (rj + __popc(mine) >= 4096) { fate = DW_FATE_NAN_ABORT; ++step; rj = -1; }        // the loop gives up (never observed)
          else rj += __popc(mine);
        }
      }
#elif DW_RAYL_REQUEUE
#pragma unroll 1
      for (int it = 0; it < DW_RAYL_REQUEUE; ++it) {
        const unsigned rm = __ballot_sync(0xffffffffu, rj >= 0);
        if (!rm) break;
        CNT(C_RAYL_ITER, 1); CNT(C_LANES_RAYL, __popc(rm));
        if (rj >= 0) {
          // ------------------------------------------------------ S6, iteration rj: isotropic k', accept with probability |e - (e.k')k'|^2
          const float4 r = DRAW_HOT(pid, step, 1u + (uint32_t)rj);
          const float ct = 1.0f - 2.0f * r.x;
          const float st_ = sqrtf(fmaxf(0.f, 1.0f - ct * ct));
          float sp, cp;
          sincospif(2.0f * r.y, &sp, &cp);
          const V3 kn = mk(st_ * cp, st_ * sp, ct);
          const V3 er = fma3(-dot(e, kn), kn, e);
          const float w = dot(er, er);
          if (r.z < w) { k = kn; e = rsqrtf(w) * er; ++step; rj = -1; }          // S9
          else if (rj + 1 >= 4096) { fate = DW_FATE_NAN_ABORT; ++step; rj = -1; } // the loop gives up (never observed)
          else ++rj;
        }
      }
      if (DW_RAYL_REQUEUE && slot >= 0 && rj >= 0) {
        // rejected: the slot waits for the next phase with the iteration number (position and time are those of the scatter point)
        poolf[W_X * kSlots + slot] = x.x; poolf[W_Y * kSlots + slot] = x.y; poolf[W_Z * kSlots + slot] = x.z;
        poolf[W_T * kSlots + slot] = t;
        pool[W_LAST * kSlots + slot] = last_tri;
        pool[W_HIST * kSlots + slot] = (int)hist;
        pool[W_BEST_SLOT * kSlots + slot] = kRaylPending - rj;
      }
#endif
      if (slot >= 0 && fate == 0xFFu && rj < 0) {
        // ---------------------------------------------------------- set up the query of the next iteration: S1 (+S3/S4 draws)
        if ((int32_t)step >= A.max_steps) {
          fate = DW_FATE_TRUNCATED;                                   // S10
        } else if (!(isfinite(x.x + x.y + x.z) && isfinite(k.x + k.y + k.z) && isfinite(e.x + e.y + e.z) && isfinite(t))) {
          fate = DW_FATE_NAN_ABORT;                                   // S11
        } else {
          float tmax = INFINITY;
          bool skip = false;
          if ((!literal) && medium >= 0) {                            // medium known: S3/S4 draws before the query
            float4 r0 = DRAW_HOT(pid, step, 0u);
            us = r0.z; uf = r0.w;
            n1 = TAB(A.tab.mat, medium, A.tab.nl_mat, A.tab.mat_l0, A.tab.mat_inv_dl, lambda);
            float La = TAB(A.tab.mat + (size_t)A.tab.n_mat * A.tab.nl_mat, medium, A.tab.nl_mat, A.tab.mat_l0, A.tab.mat_inv_dl, lambda);
            float Ls = TAB(A.tab.mat + 2 * (size_t)A.tab.n_mat * A.tab.nl_mat, medium, A.tab.nl_mat, A.tab.mat_l0, A.tab.mat_inv_dl, lambda);
            float da = -La * logf(r0.x), ds = -Ls * logf(r0.y);
            absorb_first = da < ds;
            dbulk = fminf(da, ds);
            tmax = dbulk + A.bvh.eps_len;
            // empty boxes: if the whole segment lies in triangle-free boxes of the grid, the answer is "no hit"
            if (use_grid) skip = segment_is_free(A.bvh, x, k, tmax);
          }
          poolf[W_X * kSlots + slot] = x.x; poolf[W_Y * kSlots + slot] = x.y; poolf[W_Z * kSlots + slot] = x.z;
          poolf[W_KX * kSlots + slot] = k.x; poolf[W_KY * kSlots + slot] = k.y; poolf[W_KZ * kSlots + slot] = k.z;
          poolf[W_EX * kSlots + slot] = e.x; poolf[W_EY * kSlots + slot] = e.y; poolf[W_EZ * kSlots + slot] = e.z;
          if constexpr (!kLean) poolf[W_LAMBDA * kSlots + slot] = lambda;
          poolf[W_T * kSlots + slot] = t;
          pool[W_MEDIUM * kSlots + slot] = medium;
          pool[W_LAST * kSlots + slot] = last_tri;
          pool[W_STEP * kSlots + slot] = (int)step;
          pool[W_HIST * kSlots + slot] = (int)(hist | (absorb_first ? kAbsorbFirstBit : 0u));
          pool[W_PI * kSlots + slot] = (int)(uint32_t)pi;
          poolf[W_DBULK * kSlots + slot] = dbulk;
          if constexpr (!kLean) poolf[W_N1 * kSlots + slot] = n1;
          poolf[W_US * kSlots + slot] = us;
          poolf[W_UF * kSlots + slot] = uf;
          poolf[W_BEST_T * kSlots + slot] = tmax;                     // the query starts from t_max
          pool[W_BEST_SLOT * kSlots + slot] = -1;
          st[slot] = skip ? S_PHYS : S_TRACE;                         // a skipped query is already finished: no hit
          if constexpr (kCount) { atomicAdd(&s_cnt[C_LANES_SETUP], 1ull); if (skip) atomicAdd(&s_cnt[C_SKIPPED], 1ull); }
        }
      }

      // -------------------------------------------------------------- a10: outputs and reductions
      if (fate != 0xFFu) {
        if (A.out.flags) st_out(A.out.flags + pi, fate | hist);
        if (A.out.channel) st_out(A.out.channel + pi, channel);
        if (A.out.t) st_out(A.out.t + pi, t);
        if (A.out.steps) st_out(A.out.steps + pi, step);
        if (A.out.last_tri) st_out(A.out.last_tri + pi, last_tri);
        if (A.out.x) st_out(A.out.x + pi, x.x);
        if (A.out.y) st_out(A.out.y + pi, x.y);
        if (A.out.z) st_out(A.out.z + pi, x.z);
        if (A.out.kx) { st_out(A.out.kx + pi, k.x); st_out(A.out.ky + pi, k.y); st_out(A.out.kz + pi, k.z); }
        if (A.out.ex) { st_out(A.out.ex + pi, e.x); st_out(A.out.ey + pi, e.y); st_out(A.out.ez + pi, e.z); }
        atomicAdd(&s_fate[fate & 7u], 1u);
        atomicAdd(&s_steps, (unsigned long long)step);
        st[slot] = S_EMPTY;
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
      __syncwarp();
      continue;
    }

    // ---------------------------------------------------------------- phase T: idle lanes fetch TRACE slots, then a4
    if (nQ > 0 && idle) {
      if (s0 == S_TRACE) q[__popc(t0 & lt)] = lane;
      if (s1 == S_TRACE) q[__popc(t0) + __popc(t1 & lt)] = lane + 32;
      if constexpr (kSlots > 64) { if (s2 == S_TRACE) q[__popc(t0) + __popc(t1) + __popc(t2 & lt)] = lane + 64; }
      __syncwarp();
      const int r = __popc(idle & lt);
      if (my < 0 && r < nQ) {
        my = q[r];
        V3 x = mk(poolf[W_X * kSlots + my], poolf[W_Y * kSlots + my], poolf[W_Z * kSlots + my]);
        V3 k = mk(poolf[W_KX * kSlots + my], poolf[W_KY * kSlots + my], poolf[W_KZ * kSlots + my]);
        ray_setup(ray, x, k, A.bvh);
        ts_begin(ts, poolf[W_BEST_T * kSlots + my]);
        q_exclude = pool[W_LAST * kSlots + my];
        // literal mode: every triangle counts, except right after a surface event, where a hit whose near side is not the medium the
        // photon was just sent into is an artefact of the fp32 position (G3)
        q_medium = (literal && q_exclude < 0) ? -1 : pool[W_MEDIUM * kSlots + my];
        st[my] = S_BUSY;
        if constexpr (kCount) atomicAdd(&s_cnt[C_TRACED], 1ull);
      }
      CNT(C_FETCH, 1);
      __syncwarp();
    }
    int nQ_rem = max(0, nQ - __popc(idle));
    int nReady = nP + nE;                                   // slots the physics phase could take
    int prevAct = -1;
    for (;;) {
      const bool act = my >= 0;
      const int nI = __popc(__ballot_sync(0xffffffffu, act && ts.node >= 0));
      const int nL = __popc(__ballot_sync(0xffffffffu, act && ts.node == kInLeaf));
      const int nAct = nI + nL;
      if (prevAct >= 0) nReady += prevAct - nAct;           // queries that ended in the last iteration
      prevAct = nAct;
      if (nAct == 0) break;
      if (32 - nAct >= th_fetch && (nQ_rem > 0 || nReady >= DW_TH_READY)) break;
      if (nI > 0 && nL < th_leaf) {
#if DW_NODE_REPS > 1
        // several node visits per vote while most lanes are in internal nodes: the votes are a quarter of the traversal's instructions
        const int reps = nI >= DW_NODE_REPS_MIN ? DW_NODE_REPS : 1;
        CNT(C_ITER_NODE, reps); CNT(C_LANES_NODE, nI * reps);
#pragma unroll 1
        for (int rep = 0; rep < reps; ++rep)
#endif
        if (act && ts.node >= 0) {
          step_internal(A.bvh, ray, ts, my_stack, sstride, lstack);
          if constexpr (kCount) { atomicAdd(&s_cnt[C_NODE], 1ull); ++my_visits; }
        }
      } else {
        CNT(C_ITER_LEAF, DW_TRI_REPS); CNT(C_LANES_LEAF, nL * DW_TRI_REPS);
#if DW_TRI_PAIR
        // the records of two triangles of the leaf are loaded together: one memory round trip per triangle phase, not two
        if (act && ts.node == kInLeaf) {
          const bool two = ts.tri_cur + 1 < ts.tri_end;
          TriRegs t0, t1;
          tri_load(A.bvh, ts.tri_cur, t0);
          tri_load(A.bvh, two ? ts.tri_cur + 1 : ts.tri_cur, t1);
          const float tback = (q_exclude >= 0 && q_medium >= 0) ? -8.0f * A.bvh.eps_len : 0.f;
          tri_process(ray, ts, t0, q_exclude, q_medium, tback, my_stack, sstride, lstack);
          if (two) tri_process(ray, ts, t1, q_exclude, q_medium, tback, my_stack, sstride, lstack);
          if constexpr (kCount) atomicAdd(&s_cnt[C_TRI], two ? 2ull : 1ull);
        }
#else
#if DW_TRI_REPS > 1
#pragma unroll 1
        for (int rep = 0; rep < DW_TRI_REPS; ++rep)
#endif
        if (act && ts.node == kInLeaf) {
          step_triangle(A.bvh, ray, ts, q_exclude, q_medium, my_stack, sstride, lstack);
          if constexpr (kCount) atomicAdd(&s_cnt[C_TRI], 1ull);
        }
#endif
      }
      if (act && ts.node == kDone) {                        // query finished: hand the slot to the physics phase
        if constexpr (kCount) {                             // by kind of query: first (unbounded), from a surface, from the bulk
          const int cls = q_medium < 0 ? C_Q_FRESH : (q_exclude >= 0 ? C_Q_SURF : C_Q_BULK);
          atomicAdd(&s_cnt[cls], 1ull);
          atomicAdd(&s_cnt[cls + 1], (unsigned long long)my_visits);
          if (cls != C_Q_FRESH && ts.best_slot >= 0) atomicAdd(&s_cnt[cls + 2], 1ull);
          my_visits = 0;
        }
        poolf[W_BEST_T * kSlots + my] = ts.best_t;
        pool[W_BEST_SLOT * kSlots + my] = ts.best_slot;
        st[my] = S_PHYS;
        my = -1;
      }
    }
    __syncwarp();
  }

  __syncthreads();
  if (threadIdx.x < 8 && A.hist.fate_count && s_fate[threadIdx.x]) atomicAdd((unsigned long long*)&A.hist.fate_count[threadIdx.x], (unsigned long long)s_fate[threadIdx.x]);
  if (threadIdx.x == 0 && A.hist.total_steps && s_steps) atomicAdd((unsigned long long*)A.hist.total_steps, s_steps);
  if constexpr (kCount) { if (threadIdx.x < kCounters && A.counters && s_cnt[threadIdx.x]) atomicAdd(&A.counters[threadIdx.x], s_cnt[threadIdx.x]); }
#undef CNT
}

// ------------------------------------------------------------------------------------------------ emission (f1)
// One photon per thread; the steps and draws of include/darwinopt.h "dw_emit" (Table 2).
constexpr uint32_t kEmitStep = 0xFFFFFFFFu;
__device__ __forceinline__ V3 isotropic(float u_cos, float u_phi) {
  float ct = 1.0f - 2.0f * u_cos, st = sqrtf(fmaxf(0.f, 1.0f - ct * ct)), sp, cp;
  sincospif(2.0f * u_phi, &sp, &cp);
  return mk(st * cp, st * sp, ct);
}
__device__ __forceinline__ void emit_one(const dw_source& S, uint64_t seed, const dw_photons& P, int64_t i) {
  const uint64_t pid = P.photon_id_base + (uint64_t)i;
  const float4 a = draw4(seed, pid, kEmitStep, 0u), b = draw4(seed, pid, kEmitStep, 1u), c = draw4(seed, pid, kEmitStep, 2u);
  V3 x = mk(S.centre[0], S.centre[1], S.centre[2]);
  if (S.shape == DW_SOURCE_CYLINDER) {
    float r = S.radius * sqrtf(a.x), sp, cp;
    sincospif(2.0f * a.y, &sp, &cp);
    x = mk(fmaf(r, cp, S.centre[0]), fmaf(r, sp, S.centre[1]), fmaf(S.z1 - S.z0, a.z, S.z0));
  } else if (S.shape == DW_SOURCE_BALL) {
    x = fma3(S.radius * cbrtf(a.x), isotropic(a.y, a.z), x);
  }
  const V3 k = isotropic(b.x, b.y);
  const V3 kr = cross(k, isotropic(b.z, b.w));
  V3 e, e2;
  if (dot(kr, kr) < 1e-12f) frame(k, e, e2);
  else e = unit(kr);
  const float lambda = fmaf(S.lambda_sigma * sqrtf(-2.0f * logf(c.x)), cospif(2.0f * c.y), S.lambda_mean);
  const float tau = (c.z < S.f_singlet) ? S.tau1 : S.tau3;
  const float t = fmaf(-tau, logf(c.w), S.t_start);
  float* const* o = (float* const*)&P.px;          // the eleven arrays follow each other in dw_photons
  o[0][i] = x.x; o[1][i] = x.y; o[2][i] = x.z; o[3][i] = k.x; o[4][i] = k.y; o[5][i] = k.z;
  o[6][i] = e.x; o[7][i] = e.y; o[8][i] = e.z; o[9][i] = lambda; o[10][i] = t;
}
__global__ void emit_kernel(dw_source S, uint64_t seed, dw_photons P) {
  const int64_t i = blockIdx.x * (int64_t)blockDim.x + threadIdx.x;
  if (i < P.n) emit_one(S, seed, P, i);
}
// dw_emit_sources: photon i belongs to source i / pps (many point sources per study); the source record is read through
// the read-only path (neighbouring photons share it).
__global__ void emit_sources_kernel(const dw_source* __restrict__ S, int64_t pps, uint64_t seed, dw_photons P) {
  const int64_t i = blockIdx.x * (int64_t)blockDim.x + threadIdx.x;
  if (i >= P.n) return;
  const int4* q = reinterpret_cast<const int4*>(S + i / pps);
  static_assert(sizeof(dw_source) == 64, "dw_source is read as four 128-bit words");
  union { int4 w[4]; dw_source s; } u;
  u.w[0] = __ldg(q); u.w[1] = __ldg(q + 1); u.w[2] = __ldg(q + 2); u.w[3] = __ldg(q + 3);
  emit_one(u.s, seed, P, i);
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

// ------------------------------------------------------------------------------------------------ ray cast of the mesh (dw_render)
// One pinhole-camera ray per pixel through the first-hit query: the part of the paper's "Chroma rendering" (insert of
// Fig. 1) that needs no display.  Pixel (i, j), i to the right, j downwards: d = unit(f + x r + y u) with x = 2 (i + 0.5) / w - 1,
// y = 1 - 2 (j + 0.5) / h and r, u already scaled by tan(fov / 2) (and the aspect ratio) on the host.  A warp covers an 8 x 4 pixel
// tile so that its rays stay together in the tree.  shade = round(255 |n . d|), 0 where nothing is hit.
struct DwCameraDev { float eye[3], f[3], r[3], u[3]; int w, h; };
__global__ void __launch_bounds__(128) render_kernel(DwBvh bvh, DwCameraDev cam, int32_t* __restrict__ tri, float* __restrict__ depth,
                                                     uint8_t* __restrict__ shade) {
  extern __shared__ int s_stack[];
  int lstack[kStackLocal];
  const int tiles_x = (cam.w + 15) / 16;
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const int i = (blockIdx.x % tiles_x) * 16 + (warp & 1) * 8 + (lane & 7);
  const int j = (blockIdx.x / tiles_x) * 8 + (warp >> 1) * 4 + (lane >> 3);
  if (i >= cam.w || j >= cam.h) return;
  const float x = 2.0f * ((float)i + 0.5f) / (float)cam.w - 1.0f, y = 1.0f - 2.0f * ((float)j + 0.5f) / (float)cam.h;
  const V3 d = unit(mk(fmaf(x, cam.r[0], fmaf(y, cam.u[0], cam.f[0])), fmaf(x, cam.r[1], fmaf(y, cam.u[1], cam.f[1])),
                       fmaf(x, cam.r[2], fmaf(y, cam.u[2], cam.f[2]))));
  Ray r;
  ray_setup(r, mk(cam.eye[0], cam.eye[1], cam.eye[2]), d, bvh);
  TraceState s;
  ts_begin(s, INFINITY);
  int* my = s_stack + threadIdx.x;
  while (s.node != kDone) {
    if (s.node >= 0) step_internal(bvh, r, s, my, blockDim.x, lstack);
    else step_triangle(bvh, r, s, -1, -1, my, blockDim.x, lstack);
  }
  const int64_t px = (int64_t)j * cam.w + i;
  const bool hit = s.best_slot >= 0;
  if (tri) tri[px] = hit ? (s.best_id & ~kThruSlack) : -1;
  if (depth) depth[px] = hit ? s.best_t : INFINITY;
  if (shade) {
    float v = 0.f;
    if (hit) {
      const float4* p = bvh.tris + 3 * (size_t)s.best_slot;
      const float4 a = __ldg(p), b = __ldg(p + 1), c = __ldg(p + 2);
      const V3 n = unit(cross(mk(a.w, b.x, b.y), mk(b.z, b.w, c.x)));
      v = floorf(fmaf(255.0f, fabsf(dot(n, d)), 0.5f));
    }
    shade[px] = (uint8_t)fminf(v, 255.f);
  }
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

int dw_render_impl(dw_ctx* c, const dw_camera* cam, int32_t* tri, float* depth, uint8_t* shade, cudaStream_t stream) {
  // camera basis in double precision: f = unit(forward), r = unit(f x up), u = r x f, then r and u scaled to the image half-sizes
  double f[3] = {cam->forward[0], cam->forward[1], cam->forward[2]}, up[3] = {cam->up[0], cam->up[1], cam->up[2]};
  const double fl = sqrt(f[0] * f[0] + f[1] * f[1] + f[2] * f[2]);
  if (!(fl > 0.0) || !isfinite(fl)) return dw_fail(c, DW_E_ARG, "dw_render: forward must be a finite non-zero vector");
  for (int a = 0; a < 3; ++a) f[a] /= fl;
  double r[3] = {f[1] * up[2] - f[2] * up[1], f[2] * up[0] - f[0] * up[2], f[0] * up[1] - f[1] * up[0]};
  const double rl = sqrt(r[0] * r[0] + r[1] * r[1] + r[2] * r[2]);
  const double ul = sqrt(up[0] * up[0] + up[1] * up[1] + up[2] * up[2]);
  if (!(rl > 1e-6 * ul) || !isfinite(rl)) return dw_fail(c, DW_E_ARG, "dw_render: up must be finite and not parallel to forward");
  for (int a = 0; a < 3; ++a) r[a] /= rl;
  const double u[3] = {r[1] * f[2] - r[2] * f[1], r[2] * f[0] - r[0] * f[2], r[0] * f[1] - r[1] * f[0]};
  const double th = tan(0.5 * (double)cam->fov_y_deg * 3.14159265358979323846 / 180.0), aspect = (double)cam->width / (double)cam->height;
  DwCameraDev d;
  for (int a = 0; a < 3; ++a) {
    d.eye[a] = cam->eye[a]; d.f[a] = (float)f[a]; d.r[a] = (float)(r[a] * th * aspect); d.u[a] = (float)(u[a] * th);
  }
  d.w = cam->width; d.h = cam->height;
  const int B = 128;
  const unsigned tiles = (unsigned)(((cam->width + 15) / 16) * (int64_t)((cam->height + 7) / 8));
  render_kernel<<<tiles, B, sizeof(int) * kStackShared * B, stream>>>(c->bvh, d, tri, depth, shade);
  DW_CUDA(c, cudaGetLastError());
  return DW_OK;
}

// One launch over photons [0, in->n) of `in`; n <= kMaxLaunch for the pool kernel (slot word W_PI is 32 bits).
static int launch_propagate(dw_ctx* c, const dw_photons* in, uint64_t seed, int32_t max_steps, const dw_results* out,
                            const dw_hists* hist, const dw_propagate_params* params, cudaStream_t stream,
                            unsigned long long* counters = nullptr) {
  static_assert(sizeof(PropArgs) <= 4000, "kernel parameter block too large");
  PropArgs A{};
  A.bvh = c->bvh; A.tab = c->tables; A.in = *in;
  if (out) A.out = *out;
  if (hist) A.hist = *hist;
  for (int r = 0; r < 10; ++r) {
    A.keys[2 * r] = (uint32_t)seed + (uint32_t)r * 0x9E3779B9u;
    A.keys[2 * r + 1] = (uint32_t)(seed >> 32) + (uint32_t)r * 0xBB67AE85u;
  }
  A.seed = seed; A.max_steps = max_steps; A.flags = params ? params->flags : 0u;
  const bool legacy = (A.flags & DW_PROP_LEGACY_SCHEDULER) != 0;
  A.th_phys = (params && params->th_phys > 0) ? params->th_phys : (legacy ? 12 : 8);
  A.th_leaf = (params && params->th_leaf > 0) ? params->th_leaf : 12;
  A.counters = counters;
  int B = (params && params->block_threads) ? params->block_threads : 128;
  if (B < 32 || B > 128 || (B & 31)) return dw_fail(c, DW_E_ARG, "dw_propagate: block_threads must be 32, 64, 96 or 128");
  int per_sm = 0;
  const bool films = c->tables.film != nullptr && c->tables.film_on != nullptr;
  const bool flat = DW_FLAT_TABLES && c->tables.nl_mat == 1 && c->tables.nl_surf == 1;
  if (counters && legacy) return dw_fail(c, DW_E_ARG, "dw_propagate_counters: the counters exist in the default scheduler only");
  size_t smem = legacy ? sizeof(int) * kStackShared * B : sizeof(int) * (size_t)warp_ints(flat && !films) * (B / 32);
  void (*kern)(PropArgs) = nullptr;
  if (legacy) kern = films ? propagate_kernel<true> : propagate_kernel<false>;
  else if (counters) kern = films ? (flat ? propagate_pool_kernel<true, true, true> : propagate_pool_kernel<true, false, true>)
                                  : (flat ? propagate_pool_kernel<false, true, true> : propagate_pool_kernel<false, false, true>);
  else kern = films ? (flat ? propagate_pool_kernel<true, true, false> : propagate_pool_kernel<true, false, false>)
                    : (flat ? propagate_pool_kernel<false, true, false> : propagate_pool_kernel<false, false, false>);
  DW_CUDA(c, cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, kern, B, smem));
  if (params && params->blocks_per_sm > 0) per_sm = std::min(per_sm, params->blocks_per_sm);
  if (per_sm < 1) return dw_fail(c, DW_E_CUDA, "dw_propagate: kernel does not fit on an SM");
  const int64_t per_warp = legacy ? 32 : kSlots;
  int64_t warps_needed = (in->n + per_warp - 1) / per_warp;
  int64_t blocks_needed = (warps_needed + (B / 32) - 1) / (B / 32);
  int grid = (int)std::min<int64_t>((int64_t)c->sm_count * per_sm, std::max<int64_t>(blocks_needed, 1));
  // queue head: a stream-ordered 8-byte allocation, so that launches on different streams never share one
  unsigned long long* head = nullptr;
  if (c->pool) DW_CUDA(c, cudaMallocFromPoolAsync((void**)&head, sizeof(unsigned long long), c->pool, stream));
  else DW_CUDA(c, cudaMallocAsync((void**)&head, sizeof(unsigned long long), stream));
  DW_CUDA(c, cudaMemsetAsync(head, 0, sizeof(unsigned long long), stream));
  A.queue_head = head;
  kern<<<grid, B, smem, stream>>>(A);
  cudaError_t e = cudaGetLastError();
  cudaFreeAsync(head, stream);
  if (e != cudaSuccess) return dw_fail(c, DW_E_CUDA, "propagate kernel launch failed: %s", cudaGetErrorString(e));
  c->last_grid = grid; c->last_block = B; c->last_smem = (int)smem; c->n_launches += 1;
  return DW_OK;
}

template <class T> static inline T* off(T* p, int64_t o) { return p ? p + o : p; }

int dw_propagate_impl(dw_ctx* c, const dw_photons* in, uint64_t seed, int32_t max_steps, const dw_results* out,
                      const dw_hists* hist, const dw_propagate_params* params, cudaStream_t stream) {
  constexpr int64_t kMaxLaunch = int64_t(1) << 30;
  if (in->n <= kMaxLaunch) return launch_propagate(c, in, seed, max_steps, out, hist, params, stream);
  for (int64_t o = 0; o < in->n; o += kMaxLaunch) {       // larger batches: consecutive launches over id sub-ranges
    dw_photons pi = *in;
    pi.n = std::min(kMaxLaunch, in->n - o);
    pi.photon_id_base = in->photon_id_base + (uint64_t)o;
    pi.px = off(in->px, o); pi.py = off(in->py, o); pi.pz = off(in->pz, o);
    pi.kx = off(in->kx, o); pi.ky = off(in->ky, o); pi.kz = off(in->kz, o);
    pi.ex = off(in->ex, o); pi.ey = off(in->ey, o); pi.ez = off(in->ez, o);
    pi.wavelength = off(in->wavelength, o); pi.t0 = off(in->t0, o);
    dw_results po{};
    if (out) {
      po = *out;
      po.flags = off(out->flags, o); po.channel = off(out->channel, o); po.t = off(out->t, o); po.steps = off(out->steps, o);
      po.last_tri = off(out->last_tri, o); po.x = off(out->x, o); po.y = off(out->y, o); po.z = off(out->z, o);
      po.kx = off(out->kx, o); po.ky = off(out->ky, o); po.kz = off(out->kz, o);
      po.ex = off(out->ex, o); po.ey = off(out->ey, o); po.ez = off(out->ez, o);
    }
    int rc = launch_propagate(c, &pi, seed, max_steps, out ? &po : nullptr, hist, params, stream);
    if (rc != DW_OK) return rc;
  }
  return DW_OK;
}

// launch_propagate for params == NULL, counters == NULL and no histograms, with the queue head given by the caller instead of
// allocated on the stream (dw_design_study_static).  Same kernel, block size, shared memory and grid as the allocating path.
int dw_propagate_head_impl(dw_ctx* c, const dw_photons* in, uint64_t seed, int32_t max_steps, const dw_results* out,
                           unsigned long long* head, cudaStream_t stream) {
  if (in->n <= 0) return DW_OK;
  if (in->n > (int64_t(1) << 30) || !head) return dw_fail(c, DW_E_ARG, "dw_propagate_head_impl: at most 2^30 photons and a queue head");
  PropArgs A{};
  A.bvh = c->bvh; A.tab = c->tables; A.in = *in;
  if (out) A.out = *out;
  for (int r = 0; r < 10; ++r) {
    A.keys[2 * r] = (uint32_t)seed + (uint32_t)r * 0x9E3779B9u;
    A.keys[2 * r + 1] = (uint32_t)(seed >> 32) + (uint32_t)r * 0xBB67AE85u;
  }
  A.seed = seed; A.max_steps = max_steps; A.flags = 0u;
  A.th_phys = 8; A.th_leaf = 12;
  A.counters = nullptr;
  A.queue_head = head;
  const int B = 128;
  const bool films = c->tables.film != nullptr && c->tables.film_on != nullptr;
  const bool flat = DW_FLAT_TABLES && c->tables.nl_mat == 1 && c->tables.nl_surf == 1;
  const size_t smem = sizeof(int) * (size_t)warp_ints(flat && !films) * (B / 32);
  void (*kern)(PropArgs) = films ? (flat ? propagate_pool_kernel<true, true, false> : propagate_pool_kernel<true, false, false>)
                                 : (flat ? propagate_pool_kernel<false, true, false> : propagate_pool_kernel<false, false, false>);
  int per_sm = 0;
  DW_CUDA(c, cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, kern, B, smem));
  if (per_sm < 1) return dw_fail(c, DW_E_CUDA, "dw_design_study_static: kernel does not fit on an SM");
  const int64_t warps_needed = (in->n + kSlots - 1) / kSlots;
  const int64_t blocks_needed = (warps_needed + (B / 32) - 1) / (B / 32);
  const int grid = (int)std::min<int64_t>((int64_t)c->sm_count * per_sm, std::max<int64_t>(blocks_needed, 1));
  DW_CUDA(c, cudaMemsetAsync(head, 0, sizeof(unsigned long long), stream));
  kern<<<grid, B, smem, stream>>>(A);
  cudaError_t e = cudaGetLastError();
  if (e != cudaSuccess) return dw_fail(c, DW_E_CUDA, "propagate kernel launch failed: %s", cudaGetErrorString(e));
  c->last_grid = grid; c->last_block = B; c->last_smem = (int)smem; c->n_launches += 1;
  return DW_OK;
}

int dw_propagate_counters_impl(dw_ctx* c, const dw_photons* in, uint64_t seed, int32_t max_steps, const dw_propagate_params* params,
                               uint64_t* host_out, int n_out) {
  if (in->n > (int64_t(1) << 30)) return dw_fail(c, DW_E_ARG, "dw_propagate_counters: at most 2^30 photons");
  unsigned long long* d = nullptr;
  DW_CUDA(c, cudaMalloc(&d, sizeof(unsigned long long) * kCounters));
  cudaMemset(d, 0, sizeof(unsigned long long) * kCounters);
  int rc = launch_propagate(c, in, seed, max_steps, nullptr, nullptr, params, nullptr, d);
  unsigned long long h[kCounters] = {0};
  cudaError_t e = cudaMemcpy(h, d, sizeof h, cudaMemcpyDeviceToHost);
  cudaFree(d);
  if (rc != DW_OK) return rc;
  if (e != cudaSuccess) return dw_fail(c, DW_E_CUDA, "dw_propagate_counters: %s", cudaGetErrorString(e));
  for (int i = 0; i < n_out; ++i) host_out[i] = i < kCounters ? h[i] : 0;
  return DW_OK;
}

int dw_emit_impl(dw_ctx* c, const dw_source* src, uint64_t seed, const dw_photons* out, cudaStream_t stream) {
  static_assert(offsetof(dw_photons, t0) - offsetof(dw_photons, px) == 10 * sizeof(float*), "dw_photons: eleven consecutive arrays");
  if (out->n == 0) return DW_OK;
  emit_kernel<<<(unsigned)((out->n + 255) / 256), 256, 0, stream>>>(*src, seed, *out);
  DW_CUDA(c, cudaGetLastError());
  return DW_OK;
}

int dw_emit_sources_impl(dw_ctx* c, const dw_source* d_sources, int64_t pps, uint64_t seed, const dw_photons* out, cudaStream_t stream) {
  if (out->n == 0) return DW_OK;
  emit_sources_kernel<<<(unsigned)((out->n + 255) / 256), 256, 0, stream>>>(d_sources, pps, seed, *out);
  DW_CUDA(c, cudaGetLastError());
  return DW_OK;
}

int dw_debug_philox_impl(dw_ctx* c, uint64_t seed, uint64_t base, uint32_t step, uint32_t block, int64_t n,
                         uint32_t* out_raw, float* out_u, cudaStream_t stream) {
  philox_debug_kernel<<<(unsigned)((n + 255) / 256), 256, 0, stream>>>(seed, base, step, block, n, out_raw, out_u);
  DW_CUDA(c, cudaGetLastError());
  return DW_OK;
}
