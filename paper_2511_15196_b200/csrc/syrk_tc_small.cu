// syrk_tc_small.cu -- C1 for V <= 128 (C0-C2: the covariance of the fused-kernel sizes): the centred
// particle covariance Sigma = (1/(N-1)) sum_i (phi_i - mu)(phi_i - mu)^T on tcgen05 in 3xTF32
// (BASELINE.json north_star: "the V x V covariance syrk as tcgen05/TMEM tiles in 3xTF32 split
// precision"; readings A4, R6), one launch.
//
// One CTA per 128 particles.  The 128 particles x V sites tile is read once (L2-resident at these
// sizes), centred, split hi / lo and written to shared memory in the UMMA K-major interleave layout
// with the particle index as contraction index ([32 K-chunks of 4 particles][128 site rows][16 B]).
// Both MMA operands are this one tile: D[x][y] = sum_i P[x][i] P[y][i] as 16 K-steps x 3 products
// (hi*hi + hi*lo + lo*hi) into one 128 x 128 FP32 TMEM accumulator -- 48 MMAs, a chain of K = 128,
// well inside the K = 256 bound of syrk_tc.cu for the tensor core's truncating accumulation.  The
// eight warps read it back (tcgen05.ld) and write the lower triangle of the partial tile;
// syrk_reduce_kernel (covchol.cu) sums the per-CTA partials in a fixed order.
// Replaces the FP32 SIMT syrk_partial_kernel on the product path for N >= 8192 (19 -> 11 us at C1).
#include "kernels.cuh"
#include "tcgen05.cuh"

namespace phi4 {

namespace sys {
constexpr int TILE = 128;                 // particles per CTA = contraction length
constexpr int ROWS = 128;                 // site rows of the operand tile (V <= 128, zero-padded)
constexpr int CHUNK = ROWS * 16;          // one 16-byte K-chunk of all rows
constexpr int PART = (TILE / 4) * CHUNK;  // 64 KB per hi / lo part
constexpr int THREADS = 256;
constexpr int SMEM_BYTES = 2 * PART + 64;
}  // namespace sys

__global__ void __launch_bounds__(sys::THREADS, 1)
syrk_tc_small_kernel(const float* __restrict__ phi, int N, int ld, int V,
                     const float* __restrict__ mu, float* __restrict__ partial, const Ctrl* ctrl,
                     int respect_done) {
  using namespace tc;
  using namespace sys;
  extern __shared__ __align__(1024) uint8_t smem[];
  pdl_trigger();
  uint64_t* bar = reinterpret_cast<uint64_t*>(smem + 2 * PART);
  uint32_t* tmem_slot = reinterpret_cast<uint32_t*>(bar + 1);
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  if (threadIdx.x == 0) { mbar_init(smem_u32(bar), 1); fence_mbar_init(); }
  if (warp == 0) tmem_alloc(smem_u32(tmem_slot), 128);
  tc_fence_before();
  __syncthreads();
  tc_fence_after();
  const uint32_t taddr = *tmem_slot;
  pdl_wait();
  if (respect_done && ctrl->done) {
    if (warp == 0) tmem_dealloc(taddr, 128);
    return;
  }
  const int i0 = blockIdx.x * TILE;
  // centre + split: a warp instruction covers 8 site rows x 4 K-chunks of four particles: 64
  // contiguous bytes per row from global memory (whole 32-byte sectors; the tile is L2-resident)
  // and, in shared memory, 8 x 16 B = all 32 banks per chunk (four wavefronts for 512 bytes)
  constexpr int NLD = ROWS * (TILE / 4) / THREADS;          // 16 loads per thread, all in flight
  float4 g[NLD];
#pragma unroll
  for (int k = 0; k < NLD; ++k) {
    const int e = threadIdx.x + k * THREADS;
    const int u = (e >> 5), x = 8 * (u & 15) + (e & 7), c = 4 * (u >> 4) + ((e >> 3) & 3);
    g[k] = x < V ? *reinterpret_cast<const float4*>(phi + (size_t)x * ld + i0 + 4 * c)
                 : make_float4(0.f, 0.f, 0.f, 0.f);
  }
#pragma unroll
  for (int k = 0; k < NLD; ++k) {
    const int e = threadIdx.x + k * THREADS;
    const int u = (e >> 5), x = 8 * (u & 15) + (e & 7), c = 4 * (u >> 4) + ((e >> 3) & 3);
    float4 v = make_float4(0.f, 0.f, 0.f, 0.f);
    if (x < V) {
      const float m = mu[x];
      const int i = i0 + 4 * c;                       // pad particles (i >= N) contribute zeros
      v.x = i < N ? g[k].x - m : 0.f;
      v.y = i + 1 < N ? g[k].y - m : 0.f;
      v.z = i + 2 < N ? g[k].z - m : 0.f;
      v.w = i + 3 < N ? g[k].w - m : 0.f;
    }
    float4 hi, lo;
    hi.x = tf32_rna(v.x); lo.x = v.x - hi.x;
    hi.y = tf32_rna(v.y); lo.y = v.y - hi.y;
    hi.z = tf32_rna(v.z); lo.z = v.z - hi.z;
    hi.w = tf32_rna(v.w); lo.w = v.w - hi.w;
    uint8_t* dst = smem + (size_t)c * CHUNK + (size_t)x * 16;
    *reinterpret_cast<float4*>(dst) = hi;
    *reinterpret_cast<float4*>(dst + PART) = lo;
  }
  fence_proxy_async();
  __syncthreads();
  if (threadIdx.x == 0) {
    tc_fence_after();
    const uint64_t hi_d = smem_desc(smem_u32(smem), CHUNK, 128);
    const uint64_t lo_d = hi_d + (PART >> 4);
    const uint32_t idesc = instr_desc(ROWS, ROWS);
#pragma unroll 1
    for (int ks = 0; ks < TILE / 8; ++ks) {
      const uint32_t o = (uint32_t)(2 * ks) * (CHUNK >> 4);
      tc_mma_tf32(taddr, lo_d + o, hi_d + o, idesc, ks > 0);     // small terms first
      tc_mma_tf32(taddr, hi_d + o, lo_d + o, idesc, 1);
      tc_mma_tf32(taddr, hi_d + o, hi_d + o, idesc, 1);
    }
    tc_commit(smem_u32(bar));
  }
  mbar_wait_relaxed(smem_u32(bar), 0);
  tc_fence_after();
  // warp w: TMEM lane quarter w % 4 (rows x = 32 (w % 4) + lane), column half w / 4.  The tile goes
  // through shared memory (the operand space is free once the MMAs have committed; row stride 129:
  // conflict-free both ways), so that the partial tile is written with whole 128-byte rows instead
  // of one 4-byte store per lane and row (13 x the sectors)
  float* stage = reinterpret_cast<float*>(smem);
  constexpr int SP = ROWS + 1;
  {
    const int x = (warp & 3) * 32 + lane, y0 = (warp >> 2) * 64;
    const uint32_t tl = taddr + ((uint32_t)((warp & 3) * 32) << 16) + (uint32_t)y0;
#pragma unroll
    for (int cb = 0; cb < 64; cb += 16) {
      uint32_t r[16];
      tmem_ld16(tl + (uint32_t)cb, r);
      tmem_ld_wait();
#pragma unroll
      for (int j = 0; j < 16; ++j) stage[x * SP + y0 + cb + j] = __uint_as_float(r[j]);
    }
  }
  tc_fence_before();
  __syncthreads();
  float* out = partial + (size_t)blockIdx.x * V * V;
  for (int x = warp; x < V; x += THREADS / 32)
    for (int y = lane; y <= x; y += 32) out[(size_t)x * V + y] = stage[x * SP + y];
  tc_fence_before();
  __syncthreads();
  if (warp == 0) tmem_dealloc(taddr, 128);
}

bool syrk_tc_small_supported(int V, int ld) { return V <= sys::ROWS && ld % sys::TILE == 0; }

int syrk_tc_small_nsplit(int ld) { return ld / sys::TILE; }

void launch_syrk_tc_small(const float* phi, int N, int ld, int V, const float* mu, float* partial,
                          const Ctrl* ctrl, int respect_done, cudaStream_t st) {
  static bool attr_done = false;
  if (!attr_done) {
    cudaFuncSetAttribute(syrk_tc_small_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize,
                         sys::SMEM_BYTES);
    attr_done = true;
  }
  ++g_launches;
  launch_pdl(syrk_tc_small_kernel, ld / sys::TILE, sys::THREADS, sys::SMEM_BYTES, st, phi, N, ld, V, mu,
             partial, ctrl, respect_done);
}

}  // namespace phi4
