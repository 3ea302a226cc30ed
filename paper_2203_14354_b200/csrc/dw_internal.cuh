// dw_internal.cuh -- private declarations of libdarwinopt.so (CUDA side only; the oracle shares nothing
// with this tree).  Public contract: include/darwinopt.h.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

#include <string>
#include <vector>

#include "../../include/darwinopt.h"

#define DW_VERSION 109

// ---------------------------------------------------------------------------------------------------------
// Device-side views (plain structs passed by value to kernels)
// ---------------------------------------------------------------------------------------------------------

// Optical tables.  mat: [3][n_mat][nl_mat] = refractive index, absorption length, scattering length.
// surf: [4][n_surf][nl_surf] = CUMULATIVE probabilities detect, +diffuse, +specular, +transmit (S7).
struct DwTables {
  const float* mat;
  const float* surf;
  int n_mat, nl_mat, n_surf, nl_surf;
  float mat_l0, mat_inv_dl, surf_l0, surf_inv_dl;
  // thin films on the surfaces' grid: film [3][n_surf][nl_surf] = index, extinction, thickness (nm); nullptr = none
  const float* film;
  const int32_t* film_on;
};

// 4-wide BVH node, 128 B, read as seven float4 (SoA over the four children; the eighth float4 is padding):
//   q0 = lo.x[0..3]  q1 = lo.y[0..3]  q2 = lo.z[0..3]  q3 = hi.x[0..3]  q4 = hi.y[0..3]  q5 = hi.z[0..3]
//   q6 = as_float(ref[0..3])
// ref >= 0: wide node index; ref < 0: leaf, ~ref = (first_slot << 3) | (count - 1); DW_REF_NONE = empty child.
// Traversal stack: kDwStackShared entries per thread in shared memory, kDwStackLocal more in local memory; a step
// pushes at most 3, so trees up to (kDwStackShared + kDwStackLocal) / 3 levels fit (dw_build_bvh checks).
// 8 and 12 measure the same (profiles/r01_final_c2.md, r01_captures_9_to_12_c2.md); 8 lets six lean blocks fit the 164 kB shared-memory configuration.
#ifndef DW_STACK_SHARED
#define DW_STACK_SHARED 8
#endif
constexpr int kDwStackShared = DW_STACK_SHARED;
constexpr int kDwStackLocal = 84;
#define DW_REF_NONE 0x7fffffff
// Queries read the 64-byte form of the nodes (16-bit planes) instead of the 128-byte fp32 form.  Built, correct (first-hit parity
// green) and measured on the round-2 kernel: C2 43.0 against 41.8 ms, C3 46.3 against 43.7 (profiles/r02_experiments.md): the
// decode costs more issue slots than the bytes save.  Off.
#ifndef DW_NODE_Q16
#define DW_NODE_Q16 0
#endif

// Experiment (off): 8-wide nodes, 256 B = two 4-wide records (children 0-3 and 4-7), made on the host from the 4-wide tree by pulling
// the children of the largest inner children up while at most 8 result (dw_bvh.cu widen8); a visit tests all eight boxes.  No refit.
// Measured in profiles/r02_experiments.md section 5g.
#ifndef DW_WIDE8
#define DW_WIDE8 0
#endif

// Triangle record in leaf order, 48 B, read as three float4 (Moeller-Trumbore form):
//   a = (v0.x, v0.y, v0.z, e1.x)  b = (e1.y, e1.z, e2.x, e2.y)
//   c = (e2.z, as_float(caller id), as_float(code), as_float(channel))
// code = inner | outer << 8 | surface << 16 (0xFF = no surface -> Fresnel)
struct DwBvh {
  const float4* nodes;  // [n_nodes][8]
  const float4* tris;   // [n_tri][3]
  int n_nodes;
  int n_tri;
  float eps_len;        // length tolerance tied to the fp32 spacing of the scene coordinates
  // empty-space grid (nullptr = none): cells[(z*G+y)*G+x] = inclusive cell bounds of a triangle-free box around the cell
  const uint2* cells;
  int grid_n;
  float3 grid_lo, grid_cs, grid_inv_cs;
  // the same nodes in 64 bytes (what the queries read): child planes as 16-bit steps of q_cs from q_lo, rounded outwards
  //   u0 = lo.x[0..3]  u1 = lo.y  u2 = lo.z  u3 = hi.x  u4 = hi.y  u5 = hi.z  (uint2 each: child c in the 16 bits (c & 1) of word c >> 1)
  //   then ref[0..3]
  const uint4* qnodes;  // [n_nodes][4]
  float3 q_lo, q_cs;
};

struct dw_ctx {
  int device = 0;
  int sm_count = 0;
  std::string err;
  // tables
  float* d_mat = nullptr;
  float* d_surf = nullptr;
  float* d_film = nullptr;
  int32_t* d_film_on = nullptr;
  DwTables tables{};
  bool have_mat = false, have_surf = false;
  // geometry, caller order
  int64_t n_vert = 0, n_tri = 0;
  float* d_xyz = nullptr;
  int32_t* d_idx = nullptr;
  uint32_t* d_code = nullptr;
  int32_t* d_chan = nullptr;
  bool have_geom = false;
  // BVH
  float4* d_nodes = nullptr;
  uint4* d_qnodes = nullptr;
  float4* d_tris = nullptr;
  uint2* d_cells = nullptr;
  DwBvh bvh{};
  bool built = false;
  // what dw_refit_bvh needs from the last build (dw_bvh.cu); the boxes are scratch that every refit rewrites
  struct Refit {
    int n_refs = 0, split_div = 0, grid_res = 0;
    double build_area = 0.0;      // sum of the half-areas of all child boxes as built
    int* counts = nullptr;        // [n_tri] references of the triangle
    int* offs = nullptr;          // [n_tri] its first reference
    int* slot_ref = nullptr;      // [n_refs] leaf-order slot -> reference
    float *tlo = nullptr, *thi = nullptr;   // [n_tri][3] triangle boxes
    float *rlo = nullptr, *rhi = nullptr;   // [n_refs][3] reference boxes
    unsigned* scene = nullptr;    // [6] scene bounds, order-preserving uint encoding
    std::vector<int> level_start; // wide-tree level k = nodes [level_start[k], level_start[k+1])
  } rf;
  cudaMemPool_t pool = nullptr;   // queue heads of the launches (stream-ordered, memory kept between launches)
  // launch record
  int last_grid = 0, last_block = 0, last_smem = 0;
  int64_t n_launches = 0;
  // staging for dw_propagate_host
  void* stage = nullptr;
  size_t stage_bytes = 0;
  static constexpr int kStageSlotsMax = 4;
  cudaStream_t stage_streams[kStageSlotsMax] = {nullptr, nullptr, nullptr, nullptr};
  cudaEvent_t stage_events[kStageSlotsMax] = {nullptr, nullptr, nullptr, nullptr};
};

// error helpers --------------------------------------------------------------------------------------------
int dw_fail(dw_ctx* ctx, int code, const char* fmt, ...);
#define DW_CUDA(ctx, call)                                                                       \
  do {                                                                                           \
    cudaError_t e__ = (call);                                                                    \
    if (e__ != cudaSuccess)                                                                      \
      return dw_fail((ctx), DW_E_CUDA, "%s failed: %s (%s:%d)", #call, cudaGetErrorString(e__), \
                     __FILE__, __LINE__);                                                        \
  } while (0)

// implemented in dw_bvh.cu
int dw_bvh_build_impl(dw_ctx* ctx, const dw_build_params* params, dw_build_stats* stats, cudaStream_t stream);
int dw_bvh_refit_impl(dw_ctx* ctx, const float* xyz, int on_device, dw_refit_stats* stats, cudaStream_t stream);
void dw_bvh_free(dw_ctx* ctx);   // nodes, triangle records, grid and the refit state
// implemented in dw_kernels.cu
int dw_first_hit_impl(dw_ctx* ctx, int64_t n, const float* ox, const float* oy, const float* oz, const float* dx,
                      const float* dy, const float* dz, const int32_t* exclude, int32_t* tri, float* dist,
                      cudaStream_t stream);
int dw_propagate_impl(dw_ctx* ctx, const dw_photons* in, uint64_t seed, int32_t max_steps, const dw_results* out,
                      const dw_hists* hist, const dw_propagate_params* params, cudaStream_t stream);
int dw_propagate_counters_impl(dw_ctx* ctx, const dw_photons* in, uint64_t seed, int32_t max_steps, const dw_propagate_params* params,
                               uint64_t* host_out, int n_out);
int dw_render_impl(dw_ctx* ctx, const dw_camera* cam, int32_t* tri, float* depth, uint8_t* shade, cudaStream_t stream);
int dw_emit_impl(dw_ctx* ctx, const dw_source* src, uint64_t seed, const dw_photons* out, cudaStream_t stream);
int dw_emit_sources_impl(dw_ctx* ctx, const dw_source* d_sources, int64_t photons_per_source, uint64_t seed, const dw_photons* out,
                         cudaStream_t stream);
// The default propagation kernel over in->n <= 2^30 photons with the queue head in the caller's device memory (8 bytes, zeroed here
// on the stream) instead of a stream-ordered allocation; no per-launch parameters, no histograms (dw_static.cu).
int dw_propagate_head_impl(dw_ctx* ctx, const dw_photons* in, uint64_t seed, int32_t max_steps, const dw_results* out,
                           unsigned long long* head, cudaStream_t stream);
int dw_debug_philox_impl(dw_ctx* ctx, uint64_t seed, uint64_t base, uint32_t step, uint32_t block, int64_t n,
                         uint32_t* out_raw, float* out_u, cudaStream_t stream);
// implemented in dw_api.cu
int dw_check_source(dw_ctx* ctx, const char* who, const dw_source* src);
