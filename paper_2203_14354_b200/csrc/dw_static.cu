// dw_static.cu -- dw_design_study_static (include/darwinopt.h): the design-study loop of dw_design_study for callers that may not
// allocate.  Every buffer that dw_design_study takes from the stream-ordered pool (the source table, the 15 per-photon arrays of a
// batch) and the queue head that dw_propagate allocates per launch lie in ONE file-scope device array of fixed size.  The kernels
// are the ones of the allocating path (emit_sources, the default propagation kernel, tally, tally_finish); only where their scratch
// comes from differs, so the tables come out bit for bit the same.  This file calls no cudaMalloc / cudaFree / *Async allocator.
#include <algorithm>
#include <mutex>

#include "dw_internal.cuh"

namespace {

constexpr int64_t kMaxSources = DW_STATIC_MAX_SOURCES;
constexpr int64_t kMaxPhotons = DW_STATIC_MAX_PHOTONS;
constexpr int kArrays = 15;                              // 11 photon arrays + flags, channel, t, last_tri
constexpr size_t kHeadOff = 0;                           // 8-byte queue head in a 256-byte line of its own
constexpr size_t kSrcOff = 256;
constexpr size_t kBatchOff = kSrcOff + sizeof(dw_source) * (size_t)kMaxSources;
constexpr size_t kScratchBytes = kBatchOff + sizeof(float) * kArrays * (size_t)kMaxPhotons;
static_assert(sizeof(dw_source) == 64, "dw_source is 64 bytes in DW_STATIC_SCRATCH_BYTES");
static_assert(kScratchBytes == (size_t)DW_STATIC_SCRATCH_BYTES, "the header states the size of the array");
static_assert(kBatchOff % 256 == 0, "the batch arrays start on a 256-byte line");

// One per GPU that loads this module, held until the process exits.  In host code this name is only a handle for
// cudaGetSymbolAddress: it is NOT a device address and is never passed to a kernel.
static __device__ __align__(256) unsigned char g_static_scratch[kScratchBytes];

// Device address of the array per device ordinal, looked up once per device with that device current.
constexpr int kMaxDevices = 64;
std::mutex g_mu;
unsigned char* g_addr[kMaxDevices] = {nullptr};

int scratch_of_current_device(dw_ctx* c, unsigned char** out) {
  if (c->device < 0 || c->device >= kMaxDevices)
    return dw_fail(c, DW_E_RANGE, "dw_design_study_static: device ordinal %d, at most %d are supported", c->device, kMaxDevices);
  std::lock_guard<std::mutex> lock(g_mu);
  if (!g_addr[c->device]) {
    int cur = -1;
    DW_CUDA(c, cudaGetDevice(&cur));
    if (cur != c->device) return dw_fail(c, DW_E_STATE, "dw_design_study_static: device %d is current, the context is on %d", cur, c->device);
    void* p = nullptr;
    cudaError_t e = cudaGetSymbolAddress(&p, g_static_scratch);
    if (e != cudaSuccess || !p)
      return dw_fail(c, DW_E_CUDA, "dw_design_study_static: cudaGetSymbolAddress of the scratch array failed: %s", cudaGetErrorString(e));
    g_addr[c->device] = (unsigned char*)p;
  }
  *out = g_addr[c->device];
  return DW_OK;
}

}  // namespace

extern "C" int dw_design_study_static(dw_ctx* c, const dw_source* sources, int64_t ns, int64_t pps, uint64_t seed, int32_t max_steps,
                                      const dw_tally_tables* T, float quantile, float* lce, float* t90, void* stream) {
  if (!c) return DW_E_ARG;
  if (!c->built) return dw_fail(c, DW_E_STATE, "dw_design_study_static: build the BVH first");
  if (!sources || !T || ns < 1 || pps < 1 || max_steps < 0)
    return dw_fail(c, DW_E_ARG, "dw_design_study_static: null argument, n_sources < 1, photons_per_source < 1 or max_steps < 0");
  if (ns > kMaxSources)
    return dw_fail(c, DW_E_RANGE, "dw_design_study_static: %lld sources, the static scratch holds DW_STATIC_MAX_SOURCES = %lld (use dw_design_study)",
                   (long long)ns, (long long)kMaxSources);
  if (pps > kMaxPhotons)
    return dw_fail(c, DW_E_RANGE, "dw_design_study_static: %lld photons per source, the static scratch holds DW_STATIC_MAX_PHOTONS = %lld (use dw_design_study)",
                   (long long)pps, (long long)kMaxPhotons);
  if ((lce || t90) && !(quantile > 0.f && quantile <= 1.f)) return dw_fail(c, DW_E_ARG, "dw_design_study_static: quantile outside (0, 1]");
  int rc = DW_OK;
  for (int64_t i = 0; i < ns && rc == DW_OK; ++i) rc = dw_check_source(c, "dw_design_study_static", sources + i);
  if (rc) return rc;
  DW_CUDA(c, cudaSetDevice(c->device));
  unsigned char* base = nullptr;
  rc = scratch_of_current_device(c, &base);
  if (rc) return rc;
  cudaStream_t s = (cudaStream_t)stream;
  unsigned long long* head = (unsigned long long*)(base + kHeadOff);
  dw_source* d_src = (dw_source*)(base + kSrcOff);
  float* buf = (float*)(base + kBatchOff);
  DW_CUDA(c, cudaMemcpyAsync(d_src, sources, sizeof(dw_source) * (size_t)ns, cudaMemcpyHostToDevice, s));
  const int64_t spb = std::min<int64_t>(ns, kMaxPhotons / pps);   // whole sources per batch, >= 1
  const int64_t cap = spb * pps;
  auto arr = [&](int k) { return buf + (size_t)k * cap; };
  for (int64_t s0 = 0; s0 < ns && rc == DW_OK; s0 += spb) {
    const int64_t nsb = std::min(spb, ns - s0), nb = nsb * pps;
    dw_photons ph{nb, (uint64_t)(s0 * pps), arr(0), arr(1), arr(2), arr(3), arr(4), arr(5), arr(6), arr(7), arr(8), arr(9), arr(10)};
    dw_results res{};
    res.flags = (uint32_t*)arr(11); res.channel = (int32_t*)arr(12); res.t = arr(13); res.last_tri = (int32_t*)arr(14);
    dw_tally_tables tb = *T;                              // the same tables seen from source s0 on
    if (tb.detected) tb.detected += s0 * tb.n_groups;
    if (tb.time_hist) tb.time_hist += s0 * tb.n_bins;
    if (tb.fate_by_source) tb.fate_by_source += s0 * 8;
    rc = dw_emit_sources_impl(c, d_src + s0, pps, seed, &ph, s);
    if (rc == DW_OK) rc = dw_propagate_head_impl(c, &ph, seed, max_steps, &res, head, s);
    if (rc == DW_OK) rc = dw_tally(c, &res, nb, pps, &tb, s);
  }
  if (rc == DW_OK && (lce || t90)) rc = dw_tally_finish(c, T, ns, quantile, lce, t90, s);
  return rc;
}
