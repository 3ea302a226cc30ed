// dw_probe.cu -- measured denominators for the roofline that MEASURED_PEAKS.json does not hold (BASELINE.md section 2,
// SURVEY.md 8(d) "Peaks"): issue rate of plain FP32 FMA, of plain integer ALU work, of an even mix of the two (what the
// propagation kernel issues), and the read bandwidth of an L2-resident buffer.  Register-only instruction streams pinned
// with inline PTX so that the instruction counts are known; timed with CUDA events inside the call.
#include "dw_internal.cuh"

namespace {

constexpr int kChains = 8;       // independent dependency chains per thread (latency 4 cycles, issue every cycle needs >= 4)
constexpr int kInner = 64;       // instructions per chain per outer iteration

__global__ void __launch_bounds__(256) fma_stream_kernel(int iters, float* sink) {
  float a[kChains];
  const float b = 1.0000001f, c = 1e-9f;
  for (int k = 0; k < kChains; ++k) a[k] = (float)(threadIdx.x + k);
  for (int it = 0; it < iters; ++it) {
#pragma unroll
    for (int j = 0; j < kInner; ++j) {
#pragma unroll
      for (int k = 0; k < kChains; ++k) asm volatile("fma.rn.f32 %0, %0, %1, %2;" : "+f"(a[k]) : "f"(b), "f"(c));
    }
  }
  float s = 0.f;
  for (int k = 0; k < kChains; ++k) s += a[k];
  if (s == 123.456f) *sink = s;
}

__global__ void __launch_bounds__(256) alu_stream_kernel(int iters, unsigned* sink) {
  unsigned a[kChains];
  const unsigned m = 0x9E3779B9u;
  for (int k = 0; k < kChains; ++k) a[k] = threadIdx.x * 2654435761u + k;
  for (int it = 0; it < iters; ++it) {
#pragma unroll
    for (int j = 0; j < kInner; ++j) {
#pragma unroll
      for (int k = 0; k < kChains; ++k) asm volatile("lop3.b32 %0, %0, %1, %1, 0x96;" : "+r"(a[k]) : "r"(m + k));   // xor-xor: one LOP3
    }
  }
  unsigned s = 0;
  for (int k = 0; k < kChains; ++k) s ^= a[k];
  if (s == 0xDEADBEEFu) *sink = s;
}

__global__ void __launch_bounds__(256) mix_stream_kernel(int iters, float* sink) {
  float a[kChains / 2];
  unsigned u[kChains / 2];
  const float b = 1.0000001f, c = 1e-9f;
  const unsigned m = 0x9E3779B9u;
  for (int k = 0; k < kChains / 2; ++k) { a[k] = (float)(threadIdx.x + k); u[k] = threadIdx.x * 2654435761u + k; }
  for (int it = 0; it < iters; ++it) {
#pragma unroll
    for (int j = 0; j < kInner; ++j) {
#pragma unroll
      for (int k = 0; k < kChains / 2; ++k) {
        asm volatile("fma.rn.f32 %0, %0, %1, %2;" : "+f"(a[k]) : "f"(b), "f"(c));
        asm volatile("lop3.b32 %0, %0, %1, %1, 0x96;" : "+r"(u[k]) : "r"(m + k));
      }
    }
  }
  float s = 0.f;
  for (int k = 0; k < kChains / 2; ++k) s += a[k] + (float)(u[k] & 1u);
  if (s == 123.456f) *sink = s;
}

// Every pass reads the whole buffer once, rotated by a pass-dependent offset, with volatile cache-global loads (L2, not L1), so
// that no load can be kept in a register or hoisted across passes.
__global__ void __launch_bounds__(256) l2_read_kernel(const float4* buf, size_t n_vec, int passes, float* sink) {
  float acc = 0.f;
  const size_t stride = (size_t)gridDim.x * blockDim.x, tid = blockIdx.x * (size_t)blockDim.x + threadIdx.x;
  for (int p = 0; p < passes; ++p) {
    const size_t rot = ((size_t)p * 7919u * 32u) % n_vec;
    for (size_t i = tid; i < n_vec; i += stride) {
      size_t j = i + rot;
      if (j >= n_vec) j -= n_vec;
      float x, y, z, w;
      asm volatile("ld.global.cg.v4.f32 {%0,%1,%2,%3}, [%4];" : "=f"(x), "=f"(y), "=f"(z), "=f"(w) : "l"(buf + j));
      acc += x + y + z + w;
    }
  }
  if (acc == 123.456f) *sink = acc;
}

}  // namespace

// out[0] FP32 FMA lane-instructions / s, out[1] integer ALU lane-instructions / s, out[2] lane-instructions / s of an even
// FMA + ALU mix, out[3] bytes / s read from a 32 MiB buffer that stays in L2.
extern "C" int dw_probe_peaks(dw_ctx* c, double out[4]) {
  if (!c || !out) return DW_E_ARG;
  DW_CUDA(c, cudaSetDevice(c->device));
  float* sink = nullptr;
  float4* buf = nullptr;
  cudaEvent_t e0 = nullptr, e1 = nullptr;
  const size_t bytes = 32u << 20, n_vec = bytes / sizeof(float4);
  DW_CUDA(c, cudaMalloc(&sink, 16));
  DW_CUDA(c, cudaMalloc(&buf, bytes));
  DW_CUDA(c, cudaMemset(buf, 0, bytes));
  DW_CUDA(c, cudaEventCreate(&e0)); DW_CUDA(c, cudaEventCreate(&e1));
  const int grid = c->sm_count * 8, block = 256, iters = 200;
  const double lane_instr = (double)grid * block * iters * kInner * kChains;
  float ms = 0.f;
  for (int which = 0; which < 3; ++which) {
    for (int rep = 0; rep < 2; ++rep) {                 // first repetition warms up
      DW_CUDA(c, cudaEventRecord(e0, 0));
      if (which == 0) fma_stream_kernel<<<grid, block>>>(iters, sink);
      else if (which == 1) alu_stream_kernel<<<grid, block>>>(iters, (unsigned*)sink);
      else mix_stream_kernel<<<grid, block>>>(iters, sink);
      DW_CUDA(c, cudaEventRecord(e1, 0));
      DW_CUDA(c, cudaEventSynchronize(e1));
      DW_CUDA(c, cudaEventElapsedTime(&ms, e0, e1));
    }
    out[which] = lane_instr / (ms * 1e-3);
  }
  const int passes = 50;
  for (int rep = 0; rep < 2; ++rep) {
    DW_CUDA(c, cudaEventRecord(e0, 0));
    l2_read_kernel<<<c->sm_count * 8, 256>>>(buf, n_vec, passes, sink);
    DW_CUDA(c, cudaEventRecord(e1, 0));
    DW_CUDA(c, cudaEventSynchronize(e1));
    DW_CUDA(c, cudaEventElapsedTime(&ms, e0, e1));
  }
  out[3] = (double)bytes * passes / (ms * 1e-3);
  DW_CUDA(c, cudaGetLastError());
  cudaEventDestroy(e0); cudaEventDestroy(e1); cudaFree(sink); cudaFree(buf);
  return DW_OK;
}
