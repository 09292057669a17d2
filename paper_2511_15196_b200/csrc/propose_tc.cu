// propose_tc.cu -- M1 + M2 for lattices beyond the fused kernel (V > 112, any V: the packed
// operands are zero-padded to 256 rows / 16 columns): the proposal product
//   phi'[x][i] = phi[x][i] + sum_{y<=x} (s Lc)[x][y] z[y][i]
// as a persistent tcgen05 GEMM in 3xTF32 split precision (BASELINE.json north_star: "the N x V x V
// proposal product L*z ... as tcgen05/TMEM tiles in 3xTF32 split precision"; PAPER.md:53(i), :172).
//
//   normals_split_kernel  Philox normals of one step, split hi/lo, written straight in the UMMA
//                         K-major interleave layout, stage-major: Zs[particle tile][K-stage][part]
//                         [4 chunks][128 rows][4] -- a ring stage is one contiguous 16 KB run.
//   lsplit_tiled_kernel   s*Lc split hi/lo once per temperature, stored per (site tile, K-stage):
//                         only the rows the stage can reach (lower-triangular), one run per stage.
//   propose_tc_kernel     one CTA per SM loops over (particle tile 128) x (site tile 256) output
//                         tiles, in pairs of site tiles of equal total length.  Warp 8 streams A
//                         (normals) and B (s Lc) into a 4-stage shared-memory ring with two
//                         cp.async.bulk per stage + mbarrier; warp 9 issues tcgen05.mma kind::tf32
//                         (three products per K-step into one FP32 TMEM accumulator, K-steps above
//                         the diagonal skipped, N shrunk inside the diagonal block); warps 0-7 read
//                         the accumulator with tcgen05.ld (lane = particle) and write phi' = phi + d,
//                         coalesced along particles.  The accumulator is double-buffered (2 x 256
//                         TMEM columns), so the epilogue of a tile overlaps the MMAs of the next.
// The tensor core's FP32 accumulation truncates (measured in syrk_tc.cu: -1e-4 relative over 3000
// MMAs), so one TMEM accumulator only runs over K = 1024 (384 MMAs, ~1e-5 of |d|); the epilogue
// folds the chains into round-to-nearest FP32 register sums.
// The accept step stays in accept_kernel (mutate_generic.cu): it needs whole lattice rows of phi'.
#include "kernels.cuh"
#include "philox.cuh"
#include "tcgen05.cuh"

namespace phi4 {

namespace lg {
constexpr int TILE = 128;                    // particles per output tile = TMEM lanes
constexpr int TN = 256;                      // sites per output tile = TMEM columns per buffer
constexpr int STAGES = 4;
constexpr int CHUNK_A = TILE * 16;           // one 16-byte K-chunk of 128 rows
constexpr int CHUNK_B = TN * 16;
constexpr int A_PART = 4 * CHUNK_A;          // K = 16 per stage: 4 chunks per hi / lo part
constexpr int B_PART = 4 * CHUNK_B;
constexpr int STAGE_BYTES = 2 * A_PART + 2 * B_PART;   // 48 KB
constexpr int THREADS = 320;                 // 8 epilogue warps, producer warp, MMA warp
constexpr int SUB_STAGES = 64;               // one TMEM accumulation chain covers K = 1024
constexpr int SMEM_BYTES = STAGES * STAGE_BYTES + 256;
}  // namespace lg

// z of step t for every particle, hi/lo split, stage-major interleave layout:
// float4 index (((m * nst + q / 4) * 2 + part) * 4 + q % 4) * 128 + pr, part 0 = hi, 1 = lo.
__global__ void __launch_bounds__(128)
normals_split_kernel(float4* __restrict__ Zs, int N, int ntm, int V, int Kp, int qpb,
                     uint64_t seed, uint32_t tag, uint32_t t, const Ctrl* ctrl, int respect_done) {
  pdl_enter();
  if (respect_done && ctrl->done) return;
  const int m = blockIdx.x, pr = threadIdx.x;
  const int i = m * lg::TILE + pr, nkc = Kp >> 2;
  // SFU Box-Muller (philox.cuh, R2).  Quads beyond the lattice (K padding) stay zero;
  // sites >= V inside the last quad meet zero columns.
#pragma unroll 2
  for (int qq = 0; qq < qpb; ++qq) {
    const int q = blockIdx.y * qpb + qq;
    if (q >= nkc) break;
    float z[4] = {0.f, 0.f, 0.f, 0.f};
    if (i < N && 4 * q < V) normals4_fast(seed, tag, t, (uint32_t)i, (uint32_t)q, z);
    float4 hi, lo;
    hi.x = tc::tf32_rna(z[0]); lo.x = z[0] - hi.x;
    hi.y = tc::tf32_rna(z[1]); lo.y = z[1] - hi.y;
    hi.z = tc::tf32_rna(z[2]); lo.z = z[2] - hi.z;
    hi.w = tc::tf32_rna(z[3]); lo.w = z[3] - hi.w;
    const size_t o = ((((size_t)m * (nkc >> 2) + (q >> 2)) * 2) * 4 + (q & 3)) * lg::TILE + pr;
    Zs[o] = hi;
    Zs[o + 4 * lg::TILE] = lo;
  }
}

// ---- operand layouts: one bulk copy per operand per stage ------------------------------------
// (Round 1 issued ten copies per stage -- 2 parts of normals, 2 K-steps x 2 chunks x 2 parts of
// s*Lc; the ncu source view showed the producer warp never waiting for a free stage while the
// MMA thread polled "stage full" ~30 times per stage: the copy issue was the bottleneck.)
// Normals: Zs[m][it][part][4 chunks][128 rows][4] -- 16 KB per (particle tile, stage).
// s*Lc:    Lt[tn][it][part][kk][c][nrows][4], nrows = the rows of site tile tn that K-stage it
//          can reach: 256 below the diagonal block, 256 - 16 j in its j-th stage (both K-steps of
//          a stage start at row xs = 16 it).  32 nrows floats per stage; rows above the diagonal
//          are never stored or multiplied.
__host__ __device__ inline size_t lt_tile_base(int tn) {          // floats before site tile tn
  return (size_t)8192 * 16 * ((size_t)tn * (tn - 1) / 2) + (size_t)69632 * tn;
}
__host__ __device__ inline size_t lt_stage_off(int tn, int it) {  // floats before stage it of tile tn
  const int d0 = 16 * tn;
  if (it < d0) return lt_tile_base(tn) + (size_t)it * 8192;
  const int j = it - d0;
  return lt_tile_base(tn) + (size_t)d0 * 8192 + (size_t)32 * (256 * j - 8 * j * (j - 1));
}

__global__ void lsplit_tiled_kernel(const float* __restrict__ Lc, int V, int Vn, int Kp, float s,
                                    float* __restrict__ out, const Ctrl* ctrl, int respect_done) {
  pdl_enter();
  if (respect_done && ctrl->done) return;
  const size_t idx = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (idx >= (size_t)Kp * Vn) return;
  const int y = (int)(idx / Vn), x = (int)(idx - (size_t)y * Vn);
  const int tn = x >> 8, n0 = tn << 8, it = y >> 4;
  const int rs = max(n0, 16 * it);
  if (x < rs) return;                                // above the diagonal: never multiplied
  const int nrows = n0 + 256 - rs;
  const int kk = (y >> 3) & 1, c = (y >> 2) & 1, e = y & 3;
  const float v = (x < V && y < V && y <= x) ? s * Lc[(size_t)x * V + y] : 0.f;
  const float hi = tc::tf32_rna(v), lo = tc::tf32_rna(v - hi);
  const size_t o = lt_stage_off(tn, it) + ((size_t)((kk * 2 + c) * nrows + (x - rs))) * 4 + e;
  out[o] = hi;
  out[o + (size_t)16 * nrows] = lo;                  // part stride: 2 kk x 2 c x nrows rows x 4
}

struct ProposeTcParams {
  const float* phi; float* phip;     // [V][ld]
  const float* Zs;                   // normals_split_kernel output
  const float* Lsplit;               // packed s*Lc hi | lo (tcgen05.cuh layout)
  const Ctrl* ctrl;
  int ld, V, Vn, Kp, ntm, ntn;       // Vn = V rounded up to 256 rows, Kp = V rounded up to 16
  int respect_done, pair;
};

// Tile order.  Work item w of a CTA (w = blockIdx.x, + gridDim.x, ...) is one half of a *pair* of
// site tiles (j, ntn-1-j) of one particle tile m: a pair always spans ntn+1 K-blocks of 256, so the
// CTAs stay in step, and the ceil(ntn/2) CTAs that hold the pairs of the same m at the same time
// stream the same normal tile from K = 0 upwards together -- one HBM read, the rest L2 hits
// (round 1 ran tile-index round robin: the 4 MB normal tile of a particle block at C4 was re-read
// from HBM by every one of its 16 site tiles, 39 GB per launch against 8.6 GB of operands).
// Populations with fewer tiles than SMs (pair = 0) keep one tile per CTA.
struct TileIter {
  int pair, np, nunits, ntn, u, half;
  __device__ TileIter(int ntm, int ntn_, int pair_)
      : pair(pair_), np(pair_ ? (ntn_ + 1) >> 1 : ntn_), nunits(ntm * np), ntn(ntn_),
        u(blockIdx.x), half(0) {}
  __device__ bool valid() const { return u < nunits; }
  __device__ void tile(int& m, int& n) const {
    m = u / np;
    const int j = u % np;
    n = half ? ntn - 1 - j : j;
  }
  __device__ void next() {
    const int j = u % np;
    if (pair && !half && ntn - 1 - j != j) { half = 1; return; }
    half = 0;
    u += gridDim.x;
  }
};

__global__ void __launch_bounds__(lg::THREADS, 1) propose_tc_kernel(const ProposeTcParams p) {
  using namespace tc;
  using namespace lg;
  extern __shared__ __align__(1024) uint8_t smem[];
  // programmatic dependent launch: barrier setup and the TMEM allocation run before the wait
  pdl_trigger();
  uint64_t* bars = reinterpret_cast<uint64_t*>(smem + STAGES * STAGE_BYTES);
  const uint32_t bar0 = smem_u32(bars);
  auto full = [&](int s) { return bar0 + 8u * s; };
  auto empty = [&](int s) { return bar0 + 8u * (STAGES + s); };
  auto dfull = [&](int b) { return bar0 + 8u * (2 * STAGES + b); };
  auto dempty = [&](int b) { return bar0 + 8u * (2 * STAGES + 2 + b); };
  uint32_t* tmem_slot = reinterpret_cast<uint32_t*>(bars + 2 * STAGES + 4);
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const int V = p.V, Kp = p.Kp;

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
  pdl_wait();
  if (p.respect_done && p.ctrl->done) {
    if (warp == 0) tmem_dealloc(taddr, 2 * TN);
    return;
  }

  if (warp == 8) {
    // ================================ producer: two bulk copies per stage =====================
    if (lane == 0) {
      int s = 0;
      uint32_t ph = 0;
      const int nstz = Kp >> 4;
      for (TileIter ti(p.ntm, p.ntn, p.pair); ti.valid(); ti.next()) {
        int m, tn;
        ti.tile(m, tn);
        const int n0 = tn * TN;
        const int nst = min(n0 + TN, Kp) >> 4;               // K-stages up to the tile's last row
        const float* za = p.Zs + (size_t)m * nstz * (2 * A_PART / 4);
        for (int it = 0; it < nst; ++it) {
          const uint32_t st = ring + (uint32_t)s * STAGE_BYTES;
          const int nrows = n0 + TN - max(n0, 16 * it);      // rows of the s*Lc block of this stage
          const uint32_t bbytes = 128u * (uint32_t)nrows;    // 2 parts x 2 kk x 2 c x nrows x 16 B
          mbar_wait(empty(s), ph ^ 1);
          mbar_expect_tx(full(s), 2 * A_PART + bbytes);
          bulk_g2s(st, za + (size_t)it * (2 * A_PART / 4), 2 * A_PART, full(s));
          bulk_g2s(st + 2 * A_PART, p.Lsplit + lt_stage_off(tn, it), bbytes, full(s));
          if (++s == STAGES) { s = 0; ph ^= 1; }
        }
      }
    }
    __syncwarp();
  } else if (warp == 9) {
    // ================================ MMA issuer ==============================================
    if (lane == 0) {
      int s = 0, cnt = 0;
      uint32_t ph = 0;
      const uint64_t a_base = smem_desc(ring, CHUNK_A, 128);
      for (TileIter ti(p.ntm, p.ntn, p.pair); ti.valid(); ti.next()) {
        int m, tn;
        ti.tile(m, tn);
        const int n0 = tn * TN;
        const int nst = min(n0 + TN, Kp) >> 4;
        for (int it0 = 0; it0 < nst; it0 += SUB_STAGES, ++cnt) {
          const int buf = cnt & 1;
          mbar_wait(dempty(buf), ((cnt >> 1) & 1) ^ 1);
          tc_fence_after();
          const uint32_t dbase = taddr + (uint32_t)(buf * TN);
          const int it1 = min(nst, it0 + SUB_STAGES);
          for (int it = it0; it < it1; ++it) {
            mbar_wait(full(s), ph);
            tc_fence_after();
            const uint32_t so = (uint32_t)s * (STAGE_BYTES >> 4);
            // both K-steps of a stage reach the same rows (xs = 16 it); the block sits packed in
            // the stage as [part][kk][c][nrows][16 B], so LBO and the part stride follow nrows
            const int rowstart = max(n0, 16 * it), nrows = n0 + TN - rowstart;
            const uint32_t idesc = instr_desc(TILE, nrows);
            const uint32_t d = dbase + (uint32_t)(rowstart - n0);
            const uint64_t b_st = smem_desc(ring + 2 * A_PART, (uint32_t)nrows * 16u, 128) + so;
#pragma unroll
            for (int kk = 0; kk < 2; ++kk) {
              const uint64_t a_hi = a_base + so + (uint32_t)(2 * kk) * (CHUNK_A >> 4);
              const uint64_t a_lo = a_hi + (A_PART >> 4);
              const uint64_t b_hi = b_st + (uint32_t)(2 * kk * nrows);
              const uint64_t b_lo = b_hi + (uint32_t)(4 * nrows);
              // The first K-step of a chain overwrites the accumulator.  Only the chain that ends
              // in the diagonal block has shrunk K-steps, and it starts with a full-width one
              // (n0 is a multiple of 256 <= 16 it0 whenever it0 > 0), so no column is left stale.
              tc_mma_tf32(d, a_lo, b_hi, idesc, (it != it0) || kk);
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
    // ================================ epilogue: phi' = phi + sum of chains ====================
    // warp w: TMEM lane quarter w % 4 (32 particles), column half w / 4 (128 sites)
    int cnt = 0;
    const int Q = warp & 3, hc = warp >> 2;
    const uint32_t tlane = taddr + ((uint32_t)(Q * 32) << 16);
    for (TileIter ti(p.ntm, p.ntn, p.pair); ti.valid(); ti.next()) {
      int m, tn;
      ti.tile(m, tn);
      const int n0 = tn * TN;
      const int nst = min(n0 + TN, Kp) >> 4;
      const size_t col = (size_t)m * TILE + Q * 32 + lane;
      const int x0 = n0 + hc * 128;
      if (nst <= SUB_STAGES) {
        // one chain: phi does not depend on the product, so all 128 loads of this warp's columns
        // are issued BEFORE the wait for the accumulator -- their HBM latency hides behind the
        // MMAs of the tile (issued after the wait, 8 batches x ~1.5 us made a short tile's
        // epilogue longer than the next tile's MMAs)
        const int buf = cnt & 1;
        float f[128];
#pragma unroll
        for (int j = 0; j < 128; ++j)
          f[j] = (x0 + j < V) ? p.phi[(size_t)(x0 + j) * p.ld + col] : 0.f;
        mbar_wait_relaxed(dfull(buf), (cnt >> 1) & 1);
        tc_fence_after();
#pragma unroll
        for (int cb = 0; cb < 128; cb += 32) {
          uint32_t r0[16], r1[16];
          tmem_ld16(tlane + (uint32_t)(buf * TN + hc * 128 + cb), r0);
          tmem_ld16(tlane + (uint32_t)(buf * TN + hc * 128 + cb + 16), r1);
          tmem_ld_wait();
#pragma unroll
          for (int jj = 0; jj < 16; ++jj)
            if (x0 + cb + jj < V)
              p.phip[(size_t)(x0 + cb + jj) * p.ld + col] = f[cb + jj] + __uint_as_float(r0[jj]);
#pragma unroll
          for (int jj = 0; jj < 16; ++jj)
            if (x0 + cb + 16 + jj < V)
              p.phip[(size_t)(x0 + cb + 16 + jj) * p.ld + col] = f[cb + 16 + jj] + __uint_as_float(r1[jj]);
        }
        tc_fence_before();
        __syncwarp();
        if (lane == 0) mbar_arrive(dempty(buf));
        ++cnt;
      } else {
        float acc[128];
#pragma unroll
        for (int j = 0; j < 128; ++j) acc[j] = 0.f;
        for (int it0 = 0; it0 < nst; it0 += SUB_STAGES, ++cnt) {
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
#pragma unroll
        for (int cb = 0; cb < 128; cb += 16) {
          float f[16];
#pragma unroll
          for (int jj = 0; jj < 16; ++jj)
            f[jj] = (x0 + cb + jj < V) ? p.phi[(size_t)(x0 + cb + jj) * p.ld + col] : 0.f;
#pragma unroll
          for (int jj = 0; jj < 16; ++jj)
            if (x0 + cb + jj < V) p.phip[(size_t)(x0 + cb + jj) * p.ld + col] = f[jj] + acc[cb + jj];
        }
      }
    }
  }
  tc_fence_before();
  __syncthreads();
  if (warp == 0) tmem_dealloc(taddr, 2 * TN);
}

bool propose_tc_supported(int V) { return V > 112; }

static int num_sms_cached() {
  static int n = 0;
  if (!n) {
    int dev = 0;
    cudaGetDevice(&dev);
    cudaDeviceGetAttribute(&n, cudaDevAttrMultiProcessorCount, dev);
  }
  return n;
}

// s*Lc split hi / lo in the tiled layout propose_tc_kernel streams (lt_stage_off)
void launch_propose_lsplit(const float* Lc, int V, int ld, float s, float* Lsplit, const Ctrl* ctrl,
                           int respect_done, cudaStream_t st) {
  (void)ld;
  int Vn, Kp;
  propose_tc_dims(V, &Vn, &Kp);
  ++g_launches;
  launch_pdl(lsplit_tiled_kernel, (unsigned)(((size_t)Kp * Vn + 255) / 256), 256, 0, st, Lc, V, Vn,
             Kp, s, Lsplit, ctrl, respect_done);
}

void propose_tc_dims(int V, int* Vn, int* Kp) {
  *Vn = round_up(V, lg::TN);
  *Kp = round_up(V, 16);
}

size_t propose_tc_zsplit_floats(int V, int ld) { return (size_t)2 * round_up(V, 16) * ld; }

size_t propose_tc_lsplit_floats(int V) {
  return lt_tile_base(round_up(V, lg::TN) / lg::TN);
}

void launch_normals_split(float* Zs, int N, int ld, int V, uint64_t seed, uint32_t tag, uint32_t t,
                          const Ctrl* ctrl, int respect_done, cudaStream_t st) {
  const int Kp = round_up(V, 16);
  // quads per thread: one quad per block made 1 M blocks at C4 (block-launch-rate bound); a small
  // population keeps one quad per thread so that the grid still fills the GPU
  int qpb = (ld / lg::TILE) * (Kp / 4) / (148 * 16);
  qpb = qpb < 1 ? 1 : qpb > 8 ? 8 : qpb;
  dim3 grid(ld / lg::TILE, (Kp / 4 + qpb - 1) / qpb);
  ++g_launches;
  launch_pdl(normals_split_kernel, grid, 128, 0, st, reinterpret_cast<float4*>(Zs), N, ld / lg::TILE, V, Kp,
             qpb, seed, tag, t, ctrl, respect_done);
}

void launch_propose_tc(const float* phi, float* phip, const float* Zs, const float* Lsplit, int ld,
                       int V, const Ctrl* ctrl, int respect_done, cudaStream_t st) {
  static bool attr_done = false;
  if (!attr_done) {
    cudaFuncSetAttribute(propose_tc_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize,
                         lg::SMEM_BYTES);
    attr_done = true;
  }
  const int num_sms = num_sms_cached();
  ProposeTcParams p;
  p.phi = phi; p.phip = phip; p.Zs = Zs; p.Lsplit = Lsplit; p.ctrl = ctrl;
  p.ld = ld; p.V = V;
  propose_tc_dims(V, &p.Vn, &p.Kp);
  p.ntm = ld / lg::TILE; p.ntn = p.Vn / lg::TN; p.respect_done = respect_done;
  p.pair = p.ntm * p.ntn > num_sms;
  const int nunits = p.ntm * (p.pair ? (p.ntn + 1) / 2 : p.ntn);
  const int grid = nunits < num_sms ? nunits : num_sms;
  ++g_launches;
  launch_pdl(propose_tc_kernel, grid, lg::THREADS, lg::SMEM_BYTES, st, p);
}

}  // namespace phi4
