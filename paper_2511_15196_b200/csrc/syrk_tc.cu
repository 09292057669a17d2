// syrk_tc.cu -- C1 for lattices beyond the single-CTA sizes (V > 112; operands zero-padded to
// 256 rows and 256 particles): the centred particle covariance
//   Sigma = (1/(N-1)) sum_i (phi_i - mu)(phi_i - mu)^T
// as a tcgen05 GEMM in three-product split precision (BASELINE.json north_star: "the V x V
// covariance syrk as tcgen05/TMEM tiles in 3xTF32 split precision"; readings A4, R6).
// Operand format, template parameter F16 (as in propose_tc.cu): false = 3xTF32; true (default) =
// 3xFP16 with a power-of-two scale c = 2^(11 - e), e = floor(log2 of a bound on max |phi - mu|)
// taken on the device (mean_kernel also returns max_i |phi[x][i]|; syrk_scale_kernel) -- the same
// 11-bit significands, K = 16 per MMA instead of 8, half the operand bytes; the epilogue multiplies
// the FP32 sums by the exact 1 / c^2.
//
//   centre_split_kernel  phi[x][i] - mu[x] -> hi/lo parts in the UMMA K-major interleave layout
//                        with the particle index as contraction index: 16-byte chunks of 4 (TF32)
//                        or 8 (FP16) consecutive particles, tile-major: Ps[x / 128][chunk][part]
//                        [x % 128] -- the four chunks of a ring stage of one 128-row tile, hi and
//                        lo, are ONE contiguous 16 KB run.  Transposed through shared memory:
//                        coalesced both ways.
//   syrk_tc_kernel       work item = (lower-triangular 128 x 256 output tile, K split).  Warp 8
//                        streams a stage with three bulk copies (the row tile, the two column
//                        tiles; sixteen 2-4 KB copies with the part-major layout it replaces kept
//                        the tensor pipe at 68 %) into a 4-stage ring, warp 9 issues tcgen05.mma
//                        (hi*hi + hi*lo + lo*hi, two N = 128 halves, into one FP32 TMEM accumulator).  The tensor core's FP32 accumulation
//                        truncates: over the 1e5-term sums of a covariance that is a -1e-4
//                        relative bias (measured), so an accumulator only runs over 16 stages
//                        (96 MMAs: K = 256 or 512); warps 0-7 then fold it into round-to-nearest
//                        FP32 register sums (tcgen05.ld, double-buffered TMEM) and write the
//                        partial tile once.
//   syrk_reduce_kernel   (covchol.cu) sums the K-split partials in a fixed order, scales by
//                        1/(N-1) and mirrors the lower triangle.
#include <cuda_fp16.h>

#include "kernels.cuh"
#include "tcgen05.cuh"

namespace phi4 {

namespace sy {
constexpr int TM = 128, TN = 256, STAGES = 4;
constexpr int CHUNK_A = TM * 16, CHUNK_B = TN * 16;
constexpr int A_PART = 4 * CHUNK_A, B_PART = 4 * CHUNK_B;       // 4 chunks per stage: K = 16 / 32
constexpr int STAGE_BYTES = 2 * A_PART + 2 * B_PART;            // 48 KB
constexpr int THREADS = 320;          // 8 epilogue warps, producer warp, MMA warp
constexpr int SUB_STAGES = 16;        // TMEM accumulation chain: 16 stages (96 MMAs) per flush
constexpr int S_TOP = 11;             // FP16: the bound on max |phi - mu| scaled into [2^11, 2^12)
constexpr int SMEM_BYTES = STAGES * STAGE_BYTES + 256;
}  // namespace sy

// c and 1 / c^2 from the per-site bounds amax[x] >= max_i |phi[x][i] - mu[x]| (one small block)
__global__ void __launch_bounds__(256) syrk_scale_kernel(const float* __restrict__ amax, int V,
                                                         float* __restrict__ slot, const Ctrl* ctrl,
                                                         int respect_done) {
  if (respect_done && ctrl->done) return;
  __shared__ float red[8];
  float m = 0.f;
  for (int x = threadIdx.x; x < V; x += blockDim.x) m = fmaxf(m, amax[x]);
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) m = fmaxf(m, __shfl_xor_sync(0xffffffffu, m, o));
  if ((threadIdx.x & 31) == 0) red[threadIdx.x >> 5] = m;
  __syncthreads();
  if (threadIdx.x == 0) {
    for (int w = 1; w < 8; ++w) m = fmaxf(m, red[w]);
    const float c = (m > 0.f && isfinite(m)) ? ldexpf(1.f, sy::S_TOP - ilogbf(m)) : 1.f;
    slot[0] = c;
    slot[1] = 1.0f / (c * c);
  }
}

// (as split_f16x2 in propose_tc.cu: packed conversions on the ALU pipe)
__device__ __forceinline__ void syrk_split_f16x2(float a, float b, uint32_t& hi, uint32_t& lo) {
  const __half2 h = __floats2half2_rn(a, b);
  const float2 f = __half22float2(h);
  const __half2 l = __floats2half2_rn(a - f.x, b - f.y);
  hi = *reinterpret_cast<const uint32_t*>(&h);
  lo = *reinterpret_cast<const uint32_t*>(&l);
}

// Block = 32 sites x 128 particles.  Pad particles (i >= N) contribute exact zeros.
template <bool F16>
__global__ void __launch_bounds__(256)
centre_split_kernel(const float* __restrict__ phi, int N, int ld, int V, int Vn, int ldp,
                    const float* __restrict__ mu, uint4* __restrict__ Ps, const float* __restrict__ slot,
                    const Ctrl* ctrl, int respect_done) {
  if (respect_done && ctrl->done) return;
  __shared__ float tile[32][129];
  const int x0 = blockIdx.y * 32, i0 = blockIdx.x * 128;
  const float c = F16 ? slot[0] : 1.f;
  for (int e = threadIdx.x; e < 32 * 128; e += 256) {
    const int xr = e >> 7, ic = e & 127;
    const int i = i0 + ic, x = x0 + xr;
    tile[xr][ic] = (i < N && x < V) ? c * (phi[(size_t)x * ld + i] - mu[x]) : 0.f;   // zero padding
  }
  __syncthreads();
  constexpr int CW = F16 ? 8 : 4, CSH = F16 ? 3 : 2;     // particles per 16-byte chunk
  const size_t nkc = (size_t)(ldp >> CSH);               // chunks per row
  for (int e = threadIdx.x; e < 32 * (128 / CW); e += 256) {
    const int kc = e >> 5, xr = e & 31;                  // lanes along x: 512 B contiguous stores
    uint4 hi, lo;
    if constexpr (F16) {
      float v[8];
#pragma unroll
      for (int j = 0; j < 8; ++j) v[j] = tile[xr][8 * kc + j];
      syrk_split_f16x2(v[0], v[1], hi.x, lo.x);
      syrk_split_f16x2(v[2], v[3], hi.y, lo.y);
      syrk_split_f16x2(v[4], v[5], hi.z, lo.z);
      syrk_split_f16x2(v[6], v[7], hi.w, lo.w);
    } else {
      float v[4], h[4];
#pragma unroll
      for (int j = 0; j < 4; ++j) { v[j] = tile[xr][4 * kc + j]; h[j] = tc::tf32_rna(v[j]); }
      hi = make_uint4(__float_as_uint(h[0]), __float_as_uint(h[1]), __float_as_uint(h[2]), __float_as_uint(h[3]));
      lo = make_uint4(__float_as_uint(v[0] - h[0]), __float_as_uint(v[1] - h[1]), __float_as_uint(v[2] - h[2]),
                      __float_as_uint(v[3] - h[3]));
    }
    const int x = x0 + xr;
    const size_t o = (((size_t)(x >> 7) * nkc + (size_t)((i0 >> CSH) + kc)) * 2) * sy::TM + (x & (sy::TM - 1));
    Ps[o] = hi;
    Ps[o + sy::TM] = lo;
  }
}

struct SyrkTcParams {
  const float* Ps;       // centre_split_kernel output
  const float* slot;     // FP16: {c, 1 / c^2}
  float* partial;        // [nsplit][V][V]
  const Ctrl* ctrl;
  int V, Vn, nkc, ntm, nsplit, chunks_per_split, nitems;   // Vn = V rounded up to 256
  int respect_done;
};

// item -> (tile row tm, tile col tn, split z); only tiles that touch the lower triangle
__device__ __forceinline__ void syrk_item(const SyrkTcParams& p, int item, int& m0, int& n0,
                                          int& z) {
  // K range slow, tile fast: the CTAs of a wave walk the same particles in step, so the operand
  // panels they share are read from HBM once and from L2 afterwards
  const int ntiles = p.nitems / p.nsplit;
  z = item / ntiles;
  int t = item - z * ntiles;
  // enumerate tm = 0..ntm-1, tn = 0..floor((tm*128+127)/256)
  int tm = 0;
  for (;;) {
    const int last = min(tm * sy::TM + sy::TM - 1, p.V - 1);     // last real row of this tile row
    const int cnt = last / sy::TN + 1;
    if (t < cnt) break;
    t -= cnt;
    ++tm;
  }
  m0 = tm * sy::TM;
  n0 = t * sy::TN;
}

template <bool F16>
__global__ void __launch_bounds__(sy::THREADS, 1) syrk_tc_kernel(const SyrkTcParams p) {
  using namespace tc;
  using namespace sy;
  extern __shared__ __align__(1024) uint8_t smem[];
  if (p.respect_done && p.ctrl->done) return;
  uint64_t* bars = reinterpret_cast<uint64_t*>(smem + STAGES * STAGE_BYTES);
  const uint32_t bar0 = smem_u32(bars);
  auto full = [&](int s) { return bar0 + 8u * s; };
  auto empty = [&](int s) { return bar0 + 8u * (STAGES + s); };
  auto dfull = [&](int b) { return bar0 + 8u * (2 * STAGES + b); };
  auto dempty = [&](int b) { return bar0 + 8u * (2 * STAGES + 2 + b); };
  uint32_t* tmem_slot = reinterpret_cast<uint32_t*>(bars + 2 * STAGES + 4);
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const int V = p.V;

  if (warp == 8 && lane == 0) {
    for (int s = 0; s < STAGES; ++s) { mbar_init(full(s), 1); mbar_init(empty(s), 1); }
    for (int b = 0; b < 2; ++b) { mbar_init(dfull(b), 1); mbar_init(dempty(b), 8); }
    fence_mbar_init();
  }
  if (warp == 0) tmem_alloc(smem_u32(tmem_slot), 2 * TN);
  tc_fence_before();
  __syncthreads();
  tc_fence_after();
  const uint32_t taddr = *tmem_slot;
  const uint32_t ring = smem_u32(smem);
  const int nst = p.chunks_per_split >> 2;                 // stages (4 chunks) per item

  if (warp == 8) {
    if (lane == 0) {
      const size_t tile_f = (size_t)p.nkc * 2 * TM * 4;    // floats per 128-row tile
      const uint64_t keep = l2_policy_evict_last();        // a wave of CTAs shares its operand panels
      int s = 0;
      uint32_t ph = 0;
      for (int item = blockIdx.x; item < p.nitems; item += gridDim.x) {
        int m0, n0, z;
        syrk_item(p, item, m0, n0, z);
        const int kc0 = z * p.chunks_per_split;
        const float* a_src = p.Ps + (size_t)(m0 / TM) * tile_f;
        const float* b_src = p.Ps + (size_t)(n0 / TM) * tile_f;
        for (int it = 0; it < nst; ++it) {
          mbar_wait(empty(s), ph ^ 1);
          const uint32_t st = ring + (uint32_t)s * STAGE_BYTES;
          const size_t off = (size_t)(kc0 + 4 * it) * 2 * TM * 4;     // floats before this stage's chunks
          mbar_expect_tx(full(s), STAGE_BYTES);
          bulk_g2s_hint(st, a_src + off, 2 * A_PART, full(s), keep);
          bulk_g2s_hint(st + 2 * A_PART, b_src + off, 2 * A_PART, full(s), keep);
          bulk_g2s_hint(st + 4 * A_PART, b_src + tile_f + off, 2 * A_PART, full(s), keep);
          if (++s == STAGES) { s = 0; ph ^= 1; }
        }
      }
    }
    __syncwarp();
  } else if (warp == 9) {
    if (lane == 0) {
      int s = 0, cnt = 0;
      uint32_t ph = 0;
      // a tile's stage in shared memory: [chunk c][part][128 rows][16 B]; the two K-chunks of an MMA
      // are 2 CHUNK_A apart (LBO), hi and lo of a chunk CHUNK_A
      const uint64_t t_base = smem_desc(ring, 2 * CHUNK_A, 128);
      const uint32_t idesc = F16 ? instr_desc_f16(TM, TM) : instr_desc(TM, TM);
      for (int item = blockIdx.x; item < p.nitems; item += gridDim.x) {
        for (int sub = 0; sub < nst / SUB_STAGES; ++sub, ++cnt) {
          const int buf = cnt & 1;
          mbar_wait(dempty(buf), ((cnt >> 1) & 1) ^ 1);
          tc_fence_after();
          const uint32_t d = taddr + (uint32_t)(buf * TN);
          for (int it = 0; it < SUB_STAGES; ++it) {
            mbar_wait(full(s), ph);
            tc_fence_after();
            const uint32_t so = (uint32_t)s * (STAGE_BYTES >> 4);
#pragma unroll
            for (int kk = 0; kk < 2; ++kk) {
              const uint64_t a_hi = t_base + so + (uint32_t)(4 * kk) * (CHUNK_A >> 4);
              const uint64_t a_lo = a_hi + (CHUNK_A >> 4);
#pragma unroll
              for (int hb = 0; hb < 2; ++hb) {             // column tiles n0, n0 + 128
                const uint64_t b_hi = a_hi + (uint32_t)((2 + 2 * hb) * (A_PART >> 4));
                const uint64_t b_lo = b_hi + (CHUNK_A >> 4);
                const uint32_t dh = d + (uint32_t)(hb * TM);
                if constexpr (F16) {
                  tc_mma_f16(dh, a_lo, b_hi, idesc, (it | kk) != 0);
                  tc_mma_f16(dh, a_hi, b_lo, idesc, 1);
                  tc_mma_f16(dh, a_hi, b_hi, idesc, 1);
                } else {
                  tc_mma_tf32(dh, a_lo, b_hi, idesc, (it | kk) != 0);
                  tc_mma_tf32(dh, a_hi, b_lo, idesc, 1);
                  tc_mma_tf32(dh, a_hi, b_hi, idesc, 1);
                }
              }
            }
            tc_commit(empty(s));
            if (++s == STAGES) { s = 0; ph ^= 1; }
          }
          tc_commit(dfull(buf));
        }
      }
    }
    __syncwarp();
  } else {
    // epilogue warp w: TMEM lane quarter w % 4 (row block), column half w / 4
    int cnt = 0;
    const int Q = warp & 3, hc = warp >> 2;
    const uint32_t tlane = taddr + ((uint32_t)(Q * 32) << 16);
    const float inv = F16 ? p.slot[1] : 1.f;               // (exact power of two)
    for (int item = blockIdx.x; item < p.nitems; item += gridDim.x) {
      int m0, n0, z;
      syrk_item(p, item, m0, n0, z);
      float acc[128];
#pragma unroll
      for (int j = 0; j < 128; ++j) acc[j] = 0.f;
      for (int sub = 0; sub < nst / SUB_STAGES; ++sub, ++cnt) {
        const int buf = cnt & 1;
        mbar_wait_relaxed(dfull(buf), (cnt >> 1) & 1);
        tc_fence_after();
#pragma unroll
        for (int cb = 0; cb < 128; cb += 16) {
          uint32_t r[16];
          tmem_ld16(tlane + (uint32_t)(buf * TN + hc * 128 + cb), r);
          tmem_ld_wait();
#pragma unroll
          for (int jj = 0; jj < 16; ++jj) acc[cb + jj] += __uint_as_float(r[jj]);
        }
        tc_fence_before();
        __syncwarp();
        if (lane == 0) mbar_arrive(dempty(buf));
      }
      const int x = m0 + Q * 32 + lane, y0 = n0 + hc * 128;
      if (x < V) {
        float* out = p.partial + (size_t)z * V * V + (size_t)x * V + y0;
        if ((V & 3) == 0 && y0 + 128 <= V) {
#pragma unroll
          for (int j = 0; j < 128; j += 4)
            *reinterpret_cast<float4*>(out + j) =
                make_float4(acc[j] * inv, acc[j + 1] * inv, acc[j + 2] * inv, acc[j + 3] * inv);
        } else {
#pragma unroll
          for (int j = 0; j < 128; ++j)
            if (y0 + j < V) out[j] = acc[j] * inv;
        }
      }
    }
  }
  tc_fence_before();
  __syncthreads();
  if (warp == 0) tmem_dealloc(taddr, 2 * TN);
}

bool syrk_tc_supported(int V, int ld) { return V > 112 && ld >= 256; }

static int syrk_tc_tiles(int V) {
  int t = 0;
  for (int tm = 0; tm * sy::TM < V; ++tm) {
    int last = tm * sy::TM + sy::TM - 1;
    if (last > V - 1) last = V - 1;
    t += last / sy::TN + 1;
  }
  return t;
}

// Particles are padded to a whole number of accumulation chains (16 stages x 4 chunks)
static int syrk_ldp(int ld, bool f16) { return round_up(ld, f16 ? 512 : 256); }

// K split: every split is a whole number of accumulation chains; among the admissible counts (at most
// ld / V, so that the partial tiles stay small beside the operands) the one whose items fill whole
// waves of 148 CTAs best (round 1 took "about two waves": 160 items at C3, a second wave of 12).
int syrk_tc_nsplit(int V, int ld, bool f16) {
  const int nkc = syrk_ldp(ld, f16) >> (f16 ? 3 : 2), tiles = syrk_tc_tiles(V);
  const int chains = nkc / (4 * sy::SUB_STAGES);            // accumulation chains in the whole population
  int cap = ld / V;
  cap = cap < 1 ? 1 : cap > 64 ? 64 : cap;
  // best wave efficiency first, then the smallest count within 2 % of it (the partial tiles cost
  // 4 V^2 bytes per split to write and to reduce)
  double best_eff = 0.0;
  for (int ns = 1; ns <= chains && ns <= cap; ++ns) {
    if (chains % ns) continue;
    const int items = tiles * ns, waves = (items + 147) / 148;
    const double eff = (double)items / (148.0 * waves);
    if (eff > best_eff) best_eff = eff;
  }
  int best = 1;
  for (int ns = 1; ns <= chains && ns <= cap; ++ns) {
    if (chains % ns) continue;
    const int items = tiles * ns, waves = (items + 147) / 148;
    if ((double)items / (148.0 * waves) >= best_eff - 0.02) { best = ns; break; }
  }
  return best;
}

// split operand (either format: 2 Vn ldp(256) floats as TF32, Vn ldp(512) as FP16), then the per-site
// bounds (Vn floats) and the scale slot
static size_t syrk_operand_floats(int V, int ld) {
  const size_t Vn = round_up(V, sy::TN);
  const size_t a = 2 * Vn * syrk_ldp(ld, false), b = Vn * syrk_ldp(ld, true);
  return a > b ? a : b;
}
size_t syrk_tc_scratch_floats(int V, int ld) {
  return syrk_operand_floats(V, ld) + round_up(V, sy::TN) + 64;
}
float* syrk_tc_amax(float* Ps, int V, int ld) { return Ps + syrk_operand_floats(V, ld); }

void launch_syrk_tc(const float* phi, int N, int ld, int V, const float* mu, float* Ps,
                    float* partial, const Ctrl* ctrl, int respect_done, cudaStream_t st, bool f16) {
  static int num_sms = 0;
  if (!num_sms) {
    cudaFuncSetAttribute(syrk_tc_kernel<false>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                         sy::SMEM_BYTES);
    cudaFuncSetAttribute(syrk_tc_kernel<true>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                         sy::SMEM_BYTES);
    int dev = 0;
    cudaGetDevice(&dev);
    cudaDeviceGetAttribute(&num_sms, cudaDevAttrMultiProcessorCount, dev);
  }
  const int Vn = round_up(V, sy::TN), ldp = syrk_ldp(ld, f16);
  float* amax = syrk_tc_amax(Ps, V, ld);
  float* slot = amax + Vn;
  dim3 gc(ldp / 128, Vn / 32);
  if (f16) {
    ++g_launches;
    syrk_scale_kernel<<<1, 256, 0, st>>>(amax, V, slot, ctrl, respect_done);
    ++g_launches;
    centre_split_kernel<true><<<gc, 256, 0, st>>>(phi, N, ld, V, Vn, ldp, mu, reinterpret_cast<uint4*>(Ps), slot,
                                                  ctrl, respect_done);
  } else {
    ++g_launches;
    centre_split_kernel<false><<<gc, 256, 0, st>>>(phi, N, ld, V, Vn, ldp, mu, reinterpret_cast<uint4*>(Ps), slot,
                                                   ctrl, respect_done);
  }
  SyrkTcParams p;
  p.Ps = Ps; p.slot = slot; p.partial = partial; p.ctrl = ctrl; p.V = V; p.Vn = Vn;
  p.nkc = ldp >> (f16 ? 3 : 2);
  p.ntm = Vn / sy::TM;
  p.nsplit = syrk_tc_nsplit(V, ld, f16);
  p.chunks_per_split = p.nkc / p.nsplit;
  p.nitems = syrk_tc_tiles(V) * p.nsplit;
  p.respect_done = respect_done;
  const int grid = p.nitems < num_sms ? p.nitems : num_sms;
  ++g_launches;
  if (f16) syrk_tc_kernel<true><<<grid, sy::THREADS, sy::SMEM_BYTES, st>>>(p);
  else syrk_tc_kernel<false><<<grid, sy::THREADS, sy::SMEM_BYTES, st>>>(p);
}

}  // namespace phi4
