// measure.cu -- phi4_measure_peaks: the roofline denominators MEASURED_PEAKS.json does not hold
// ("TF32 and FP32-FMA peaks are not in that file -- the builder measures them first").
//   tf32   dense tcgen05.mma.cta_group::1.kind::tf32, M = 128, N = 256, K = 8 per instruction, one
//          CTA per SM issuing from shared-memory operands that never change (no loads: the
//          tensor pipe alone), two alternating TMEM accumulators.  Burst: best of a few ~10 ms
//          launches after warm-up; sustained: launches back to back for `seconds`.
//   f16    the same with kind::f16 (FP16 operands, FP32 accumulator), K = 16 per instruction.
//   ffma   FP32 fused multiply-adds, 8 independent chains per thread, 2 x 1024 threads per SM.
//   imad   the Philox round's integer work: 32 x 32 -> 64 multiplies (IMAD.WIDE) with a LOP3.
// Rates are returned per second; lane-ops count one FMA / one IMAD.WIDE as one operation.
#include <string.h>

#include "../../include/phi4smc.h"
#include "kernels.cuh"
#include "tcgen05.cuh"

namespace phi4 {

constexpr int MM_N = 256, MM_K8 = 8;
constexpr int MM_A_BYTES = 128 * 32, MM_B_BYTES = MM_N * 32;          // K = 8 tf32 = 32 B per row
constexpr int MM_SETS = 4;                                            // operand sets cycled through

template <bool F16>
__global__ void __launch_bounds__(128, 1) peak_mma_kernel(int iters, float* sink) {
  using namespace tc;
  extern __shared__ __align__(1024) uint8_t smem[];
  __shared__ uint64_t bar[2];
  __shared__ uint32_t tmem_slot;
  float* f = reinterpret_cast<float*>(smem);
  const int nfl = MM_SETS * (MM_A_BYTES + MM_B_BYTES) / 4;
  for (int i = threadIdx.x; i < nfl; i += blockDim.x) {
    uint32_t hsh = (uint32_t)i * 2654435761u + blockIdx.x * 40503u;
    // (FP16: the same bits read as pairs of halves -- exponent fields 0x3c.. / mantissa noise, all finite)
    f[i] = tf32_rna(((float)(hsh >> 8) * 5.9604644775390625e-8f - 0.5f) * 0.25f);
    if (F16) reinterpret_cast<uint32_t*>(f)[i] = 0x2c002c00u | (hsh & 0x03ff03ffu);
  }
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  if (threadIdx.x == 0) { mbar_init(smem_u32(&bar[0]), 1); mbar_init(smem_u32(&bar[1]), 1); fence_mbar_init(); }
  if (warp == 0) tmem_alloc(smem_u32(&tmem_slot), 512);
  fence_proxy_async();
  tc_fence_before();
  __syncthreads();
  tc_fence_after();
  const uint32_t taddr = tmem_slot;
  if (warp == 1 && lane == 0) {
    const uint32_t base = smem_u32(smem);
    const uint32_t idesc = F16 ? instr_desc_f16(128, MM_N) : instr_desc(128, MM_N);
    // batches alternate between two barriers and each barrier is waited on before its next commit
    // is issued, so no phase can be skipped: the queue holds at most two batches of 16 MMAs
    uint32_t ph[2] = {0, 0};
    for (int it = 0; it < iters; ++it) {
#pragma unroll
      for (int j = 0; j < 16; ++j) {
        const int set = j & (MM_SETS - 1);
        const uint64_t a = smem_desc(base + set * MM_A_BYTES, 128 * 16, 128);
        const uint64_t b = smem_desc(base + MM_SETS * MM_A_BYTES + set * MM_B_BYTES, MM_N * 16, 128);
        if (F16) tc_mma_f16(taddr + (uint32_t)((j & 1) * MM_N), a, b, idesc, (it | (j >> 1)) != 0);
        else tc_mma_tf32(taddr + (uint32_t)((j & 1) * MM_N), a, b, idesc, (it | (j >> 1)) != 0);
      }
      tc_commit(smem_u32(&bar[it & 1]));
      if (it > 0) { const int b = (it - 1) & 1; mbar_wait(smem_u32(&bar[b]), ph[b]); ph[b] ^= 1; }
    }
    { const int b = (iters - 1) & 1; mbar_wait(smem_u32(&bar[b]), ph[b]); }
    tc_fence_after();
  }
  __syncthreads();
  if (warp == 0) {
    uint32_t r[16];
    tmem_ld16(taddr + ((uint32_t)0 << 16), r);
    tmem_ld_wait();
    if (sink && __uint_as_float(r[lane & 15]) == 123456.789f) sink[blockIdx.x] = 1.f;   // keep the result live
    tc_fence_before();
  }
  __syncthreads();
  if (warp == 0) tmem_dealloc(taddr, 512);
}

__global__ void __launch_bounds__(1024, 2) peak_ffma_kernel(int iters, float* sink) {
  float a[8];
  const float x = 1.0f + 1e-7f * (float)threadIdx.x, y = 1e-3f * (float)(blockIdx.x & 7);
#pragma unroll
  for (int j = 0; j < 8; ++j) a[j] = (float)j + (float)threadIdx.x;
  for (int it = 0; it < iters; ++it) {
#pragma unroll
    for (int u = 0; u < 16; ++u) {
#pragma unroll
      for (int j = 0; j < 8; ++j) a[j] = fmaf(a[j], x, y);
    }
  }
  float s = 0.f;
#pragma unroll
  for (int j = 0; j < 8; ++j) s += a[j];
  if (s == 123456.789f) sink[0] = s;
}

__global__ void __launch_bounds__(1024, 2) peak_dfma_kernel(int iters, double* sink) {
  double a[8];
  const double x = 1.0 + 1e-12 * (double)threadIdx.x, y = 1e-3 * (double)(blockIdx.x & 7);
#pragma unroll
  for (int j = 0; j < 8; ++j) a[j] = (double)j + (double)threadIdx.x;
  for (int it = 0; it < iters; ++it) {
#pragma unroll
    for (int u = 0; u < 16; ++u) {
#pragma unroll
      for (int j = 0; j < 8; ++j) a[j] = fma(a[j], x, y);
    }
  }
  double s = 0.0;
#pragma unroll
  for (int j = 0; j < 8; ++j) s += a[j];
  if (s == 123456.789) sink[0] = s;
}

__global__ void __launch_bounds__(1024, 2) peak_imad_kernel(int iters, uint32_t* sink) {
  uint32_t a[8];
#pragma unroll
  for (int j = 0; j < 8; ++j) a[j] = threadIdx.x * 2654435761u + j + blockIdx.x;
  const uint32_t k = 0x9E3779B9u + blockIdx.x;
  for (int it = 0; it < iters; ++it) {
#pragma unroll
    for (int u = 0; u < 16; ++u) {
#pragma unroll
      for (int j = 0; j < 8; ++j) {
        const uint64_t p = (uint64_t)0xD2511F53u * (uint64_t)a[j];       // IMAD.WIDE
        a[j] = (uint32_t)(p >> 32) ^ (uint32_t)p ^ k;                     // LOP3
      }
    }
  }
  uint32_t s = 0;
#pragma unroll
  for (int j = 0; j < 8; ++j) s ^= a[j];
  if (s == 0x12345678u) sink[0] = s;
}

}  // namespace phi4

using namespace phi4;

extern "C" __attribute__((visibility("default")))
int phi4_measure_peaks(double seconds, phi4_peaks* out, void* d_scratch, size_t scratch_bytes,
                       void* cuda_stream) {
  if (!out || !d_scratch || scratch_bytes < 4096 || !(seconds > 0.0) || seconds > 30.0) return PHI4_EINVAL;
  cudaStream_t st = reinterpret_cast<cudaStream_t>(cuda_stream);
  int dev = 0, sms = 0;
  if (cudaGetDevice(&dev) != cudaSuccess) return PHI4_ECUDA;
  if (cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess || sms < 1)
    return PHI4_ECUDA;
  memset(out, 0, sizeof(*out));
  out->sms = sms;
  float* sink = reinterpret_cast<float*>(d_scratch);
  cudaEvent_t e0, e1;
  if (cudaEventCreate(&e0) != cudaSuccess || cudaEventCreate(&e1) != cudaSuccess) return PHI4_ECUDA;
  const int smem = MM_SETS * (MM_A_BYTES + MM_B_BYTES);
  cudaFuncSetAttribute(peak_mma_kernel<false>, cudaFuncAttributeMaxDynamicSharedMemorySize, smem);
  cudaFuncSetAttribute(peak_mma_kernel<true>, cudaFuncAttributeMaxDynamicSharedMemorySize, smem);
  auto timed = [&](auto launch, int reps) -> double {   // seconds for `reps` launches
    cudaEventRecord(e0, st);
    for (int r = 0; r < reps; ++r) launch();
    cudaEventRecord(e1, st);
    cudaEventSynchronize(e1);
    float ms = 0.f;
    cudaEventElapsedTime(&ms, e0, e1);
    return (double)ms * 1e-3;
  };
  // ---- tensor pipe: kind::tf32 (K = 8 per instruction) and kind::f16 (K = 16)
  for (int f16 = 0; f16 < 2; ++f16) {
    const int iters = 4096;                              // 16 MMAs each: ~5 ms per launch
    const double flop = 2.0 * 128 * MM_N * MM_K8 * (f16 ? 2.0 : 1.0) * 16.0 * iters * sms;
    auto launch = [&]() {
      ++g_launches;
      if (f16) peak_mma_kernel<true><<<sms, 128, smem, st>>>(iters, sink);
      else peak_mma_kernel<false><<<sms, 128, smem, st>>>(iters, sink);
    };
    timed(launch, 2);                                    // warm-up
    double best = 1e30;
    for (int r = 0; r < 5; ++r) { double t = timed(launch, 1); if (t < best) best = t; }
    const double t1 = timed(launch, 8) / 8.0;
    int reps = (int)((f16 ? 0.5 : 1.0) * seconds / t1) + 1;
    const double t = timed(launch, reps);
    if (f16) { out->f16_tflops_burst = flop / best * 1e-12; out->f16_tflops_sustained = flop * reps / t * 1e-12; }
    else { out->tf32_tflops_burst = flop / best * 1e-12; out->tf32_tflops_sustained = flop * reps / t * 1e-12; }
  }
  // ---- FP32 FMA and integer multiply lanes
  {
    const int iters = 2048, grid = 2 * sms;
    const double ops = 8.0 * 16.0 * iters * 1024.0 * grid;
    auto lf = [&]() { ++g_launches; peak_ffma_kernel<<<grid, 1024, 0, st>>>(iters, sink); };
    auto li = [&]() { ++g_launches; peak_imad_kernel<<<grid, 1024, 0, st>>>(iters, reinterpret_cast<uint32_t*>(sink)); };
    timed(lf, 2);
    double best = 1e30;
    for (int r = 0; r < 5; ++r) { double t = timed(lf, 1); if (t < best) best = t; }
    out->ffma_tlaneops = ops / best * 1e-12;
    timed(li, 2);
    best = 1e30;
    for (int r = 0; r < 5; ++r) { double t = timed(li, 1); if (t < best) best = t; }
    out->imad_wide_tlaneops = ops / best * 1e-12;
    // FP64 FMA rate (half the FP32 rate on a B200: 64 lanes per SM)
    const int itd = 64;
    const double opsd = 8.0 * 16.0 * itd * 1024.0 * grid;
    auto ld = [&]() { ++g_launches; peak_dfma_kernel<<<grid, 1024, 0, st>>>(itd, reinterpret_cast<double*>(sink)); };
    timed(ld, 2);
    best = 1e30;
    for (int r = 0; r < 5; ++r) { double t = timed(ld, 1); if (t < best) best = t; }
    out->dfma_tlaneops = opsd / best * 1e-12;
  }
  cudaEventDestroy(e0);
  cudaEventDestroy(e1);
  return cudaGetLastError() == cudaSuccess ? PHI4_OK : PHI4_ECUDA;
}
