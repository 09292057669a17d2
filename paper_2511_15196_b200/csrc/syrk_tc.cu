// syrk_tc.cu -- C1 for lattices beyond the single-CTA sizes (V > 112; operands zero-padded to
// 256 rows and 256 particles): the centred particle covariance
//   Sigma = (1/(N-1)) sum_i (phi_i - mu)(phi_i - mu)^T
// as a tcgen05 GEMM in 3xTF32 split precision (BASELINE.json north_star: "the V x V covariance
// syrk as tcgen05/TMEM tiles in 3xTF32 split precision"; readings A4, R6).
//
//   centre_split_kernel  phi[x][i] - mu[x] -> hi/lo TF32 parts in the UMMA K-major interleave
//                        layout with the particle index as contraction index:
//                        Ps[part][i / 4][x][i % 4]  (a 128-row slice of one K-chunk is 2 KB
//                        contiguous).  Transposed through shared memory: coalesced both ways.
//   syrk_tc_kernel       work item = (lower-triangular 128 x 256 output tile, K split).  Warp 8
//                        streams both operand slices of a K = 16 stage with cp.async.bulk into a
//                        4-stage ring, warp 9 issues tcgen05.mma kind::tf32 (hi*hi + hi*lo + lo*hi
//                        into one FP32 TMEM accumulator).  The tensor core's FP32 accumulation
//                        truncates: over the 1e5-term sums of a covariance that is a -1e-4
//                        relative bias (measured), so an accumulator only runs over K = 256
//                        (96 MMAs); warps 0-7 then fold it into round-to-nearest FP32 register
//                        sums (tcgen05.ld, double-buffered TMEM) and write the partial tile once.
//   syrk_reduce_kernel   (covchol.cu) sums the K-split partials in a fixed order, scales by
//                        1/(N-1) and mirrors the lower triangle.
#include "kernels.cuh"
#include "tcgen05.cuh"

namespace phi4 {

namespace sy {
constexpr int TM = 128, TN = 256, STAGES = 4;
constexpr int CHUNK_A = TM * 16, CHUNK_B = TN * 16;
constexpr int A_PART = 4 * CHUNK_A, B_PART = 4 * CHUNK_B;       // K = 16 per stage
constexpr int STAGE_BYTES = 2 * A_PART + 2 * B_PART;            // 48 KB
constexpr int THREADS = 320;          // 8 epilogue warps, producer warp, MMA warp
constexpr int SUB_STAGES = 16;        // TMEM accumulation chain: K = 256 per flush
constexpr int SMEM_BYTES = STAGES * STAGE_BYTES + 256;
}  // namespace sy

// Block = 32 sites x 128 particles.  Pad particles (i >= N) contribute exact zeros.
__global__ void __launch_bounds__(256)
centre_split_kernel(const float* __restrict__ phi, int N, int ld, int V, int Vn, int ldp,
                    const float* __restrict__ mu, float4* __restrict__ Ps, const Ctrl* ctrl,
                    int respect_done) {
  if (respect_done && ctrl->done) return;
  __shared__ float tile[32][129];
  const int x0 = blockIdx.y * 32, i0 = blockIdx.x * 128;
  for (int e = threadIdx.x; e < 32 * 128; e += 256) {
    const int xr = e >> 7, ic = e & 127;
    const int i = i0 + ic, x = x0 + xr;
    tile[xr][ic] = (i < N && x < V) ? phi[(size_t)x * ld + i] - mu[x] : 0.f;   // zero padding
  }
  __syncthreads();
  const size_t part = (size_t)(ldp >> 2) * Vn;           // float4s per hi / lo part
  for (int e = threadIdx.x; e < 32 * 32; e += 256) {
    const int kc = e >> 5, xr = e & 31;                  // lanes along x: 512 B contiguous stores
    float4 hi, lo;
    const float v0 = tile[xr][4 * kc], v1 = tile[xr][4 * kc + 1], v2 = tile[xr][4 * kc + 2],
                v3 = tile[xr][4 * kc + 3];
    hi.x = tc::tf32_rna(v0); lo.x = v0 - hi.x;
    hi.y = tc::tf32_rna(v1); lo.y = v1 - hi.y;
    hi.z = tc::tf32_rna(v2); lo.z = v2 - hi.z;
    hi.w = tc::tf32_rna(v3); lo.w = v3 - hi.w;
    const size_t o = (size_t)((i0 >> 2) + kc) * Vn + x0 + xr;
    Ps[o] = hi;
    Ps[part + o] = lo;
  }
}

struct SyrkTcParams {
  const float* Ps;       // centre_split_kernel output
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
  const int V = p.V, Vn = p.Vn;

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
  const int nst = p.chunks_per_split >> 2;                 // K = 16 stages per item

  if (warp == 8) {
    if (lane == 0) {
      const size_t part = (size_t)p.nkc * Vn * 4;          // floats per hi / lo part
      int s = 0;
      uint32_t ph = 0;
      for (int item = blockIdx.x; item < p.nitems; item += gridDim.x) {
        int m0, n0, z;
        syrk_item(p, item, m0, n0, z);
        const int kc0 = z * p.chunks_per_split;
        for (int it = 0; it < nst; ++it) {
          mbar_wait(empty(s), ph ^ 1);
          const uint32_t st = ring + (uint32_t)s * STAGE_BYTES;
          mbar_expect_tx(full(s), STAGE_BYTES);
#pragma unroll
          for (int c = 0; c < 4; ++c) {
            const size_t row = (size_t)(kc0 + 4 * it + c) * Vn;
#pragma unroll
            for (int h = 0; h < 2; ++h) {
              const float* base = p.Ps + (size_t)h * part + row * 4;
              bulk_g2s(st + (uint32_t)h * A_PART + (uint32_t)c * CHUNK_A, base + (size_t)m0 * 4,
                       CHUNK_A, full(s));
              bulk_g2s(st + 2 * A_PART + (uint32_t)h * B_PART + (uint32_t)c * CHUNK_B,
                       base + (size_t)n0 * 4, CHUNK_B, full(s));
            }
          }
          if (++s == STAGES) { s = 0; ph ^= 1; }
        }
      }
    }
    __syncwarp();
  } else if (warp == 9) {
    if (lane == 0) {
      int s = 0, cnt = 0;
      uint32_t ph = 0;
      const uint64_t a_base = smem_desc(ring, CHUNK_A, 128);
      const uint64_t b_base = smem_desc(ring + 2 * A_PART, CHUNK_B, 128);
      const uint32_t idesc = instr_desc(TM, TN);
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
              const uint64_t a_hi = a_base + so + (uint32_t)(2 * kk) * (CHUNK_A >> 4);
              const uint64_t a_lo = a_hi + (A_PART >> 4);
              const uint64_t b_hi = b_base + so + (uint32_t)(2 * kk) * (CHUNK_B >> 4);
              const uint64_t b_lo = b_hi + (B_PART >> 4);
              tc_mma_tf32(d, a_lo, b_hi, idesc, (it | kk) != 0);
              tc_mma_tf32(d, a_hi, b_lo, idesc, 1);
              tc_mma_tf32(d, a_hi, b_hi, idesc, 1);
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
            *reinterpret_cast<float4*>(out + j) = make_float4(acc[j], acc[j + 1], acc[j + 2], acc[j + 3]);
        } else {
#pragma unroll
          for (int j = 0; j < 128; ++j)
            if (y0 + j < V) out[j] = acc[j];
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

// K split: every split is a whole number of K = 256 chains; among the admissible counts (at most
// ld / V, so that the partial tiles stay small beside the operands) the one whose items fill whole
// waves of 148 CTAs best (round 1 took "about two waves": 160 items at C3, a second wave of 12).
int syrk_tc_nsplit(int V, int ld) {
  const int nkc = round_up(ld, 256) >> 2, tiles = syrk_tc_tiles(V);
  const int chains = nkc / (4 * sy::SUB_STAGES);            // K = 256 chains in the whole population
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

size_t syrk_tc_scratch_floats(int V, int ld) {
  return (size_t)2 * round_up(V, sy::TN) * round_up(ld, 256);
}

void launch_syrk_tc(const float* phi, int N, int ld, int V, const float* mu, float* Ps,
                    float* partial, const Ctrl* ctrl, int respect_done, cudaStream_t st) {
  static int num_sms = 0;
  if (!num_sms) {
    cudaFuncSetAttribute(syrk_tc_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize,
                         sy::SMEM_BYTES);
    int dev = 0;
    cudaGetDevice(&dev);
    cudaDeviceGetAttribute(&num_sms, cudaDevAttrMultiProcessorCount, dev);
  }
  const int Vn = round_up(V, sy::TN), ldp = round_up(ld, 256);
  dim3 gc(ldp / 128, Vn / 32);
  ++g_launches;
  centre_split_kernel<<<gc, 256, 0, st>>>(phi, N, ld, V, Vn, ldp, mu, reinterpret_cast<float4*>(Ps),
                                          ctrl, respect_done);
  SyrkTcParams p;
  p.Ps = Ps; p.partial = partial; p.ctrl = ctrl; p.V = V; p.Vn = Vn; p.nkc = ldp >> 2;
  p.ntm = Vn / sy::TM;
  p.nsplit = syrk_tc_nsplit(V, ld);
  p.chunks_per_split = p.nkc / p.nsplit;
  p.nitems = syrk_tc_tiles(V) * p.nsplit;
  p.respect_done = respect_done;
  const int grid = p.nitems < num_sms ? p.nitems : num_sms;
  ++g_launches;
  syrk_tc_kernel<<<grid, sy::THREADS, sy::SMEM_BYTES, st>>>(p);
}

}  // namespace phi4
