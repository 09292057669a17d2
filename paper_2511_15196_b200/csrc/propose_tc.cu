// propose_tc.cu -- M1 + M2 for lattices beyond the fused kernel (V > 112, any V: the packed
// operands are zero-padded to 256 rows / one K-stage of columns): the proposal product
//   phi'[x][i] = phi[x][i] + sum_{y<=x} (s Lc)[x][y] z[y][i]
// as a persistent tcgen05 GEMM in three-product split precision (BASELINE.json north_star: "the
// N x V x V proposal product L*z ... as tcgen05/TMEM tiles in 3xTF32 split precision";
// PAPER.md:53(i), :172).  Two operand formats, template parameter F16:
//   F16 = false  3xTF32: hi = rna_tf32(v), lo = v - hi; kind::tf32, K = 8 per instruction.
//   F16 = true   3xFP16, scaled (the default): FP16 has the SAME 11-bit significand as TF32, so
//                hi = rn_f16(c v), lo = rn_f16(c v - hi) split with the same error bounds, and
//                kind::f16 multiplies K = 16 per instruction in the same time: half the tensor
//                work and half the operand bytes.  What FP16 lacks is exponent range, hence the
//                powers of two c: normals are scaled by 2^3 (|z| < 6.7), s*Lc by 2^(12 - e) with
//                e = floor(log2 max|s Lc|) measured on the device (labsmax_kernel) -- the largest
//                entry lands in [2^12, 2^13), entries down to 2^-26 of it stay normal numbers,
//                smaller ones lose relative, not absolute, accuracy (< 2^-37 of the largest
//                entry).  The epilogue multiplies the FP32 accumulator by the exact inverse.
//
//   normals_split_kernel  Philox normals of one step, split hi/lo, written straight in the UMMA
//                         K-major interleave layout, stage-major: Zs[particle tile][K-stage][part]
//                         [4 chunks][128 rows][16 B] -- a ring stage is one contiguous 16 KB run
//                         (K = 16 TF32 or 32 FP16 columns).
//   lsplit_tiled_kernel   s*Lc split hi/lo once per temperature, stored per (site tile, K-stage):
//                         only the rows the stage can reach (lower-triangular), one run per stage.
//   propose_tc_kernel     one CTA per SM loops over (particle tile 128) x (site tile 256) output
//                         tiles, in pairs of site tiles of equal total length.  Warp 8 streams A
//                         (normals) and B (s Lc) into a 4-stage shared-memory ring with two
//                         cp.async.bulk per stage + mbarrier; warp 9 issues tcgen05.mma
//                         (three products per K-step into one FP32 TMEM accumulator, K-steps above
//                         the diagonal skipped, N shrunk inside the diagonal block); warps 0-7 read
//                         the accumulator with tcgen05.ld (lane = particle) and write phi' = phi + d,
//                         coalesced along particles.  The accumulator is double-buffered (2 x 256
//                         TMEM columns), so the epilogue of a tile overlaps the MMAs of the next.
// The tensor core's FP32 accumulation truncates (measured in syrk_tc.cu: -1e-4 relative over 3000
// MMAs), so one TMEM accumulator only runs over K = 1024 (384 / 192 MMAs, ~1e-5 of |d|); the
// epilogue folds the chains into round-to-nearest FP32 register sums.
// The accept step stays in accept_kernel (mutate_generic.cu): it needs whole lattice rows of phi'.
#include <cuda_fp16.h>

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
constexpr int A_PART = 4 * CHUNK_A;          // 4 chunks per stage and hi / lo part
constexpr int B_PART = 4 * CHUNK_B;
constexpr int STAGE_BYTES = 2 * A_PART + 2 * B_PART;   // 48 KB
// 8 epilogue warps (warpgroups 0-1), producer warp, MMA warp and 10 warps that draw the next step's
// normals (warpgroups 2-4).  The kernel is compiled for 96 registers per thread; the epilogue
// warpgroups then take 168 each (setmaxnreg.inc) out of what the other three give back (48 each):
// 8 x 168 + 12 x 48 = 20 x 96.
constexpr int THREADS = 640;
constexpr int GEN_WARP0 = 10, GEN_THREADS = THREADS - 32 * GEN_WARP0;
constexpr int REGS_EPI = 168, REGS_REST = 48;
constexpr int SMEM_BYTES = STAGES * STAGE_BYTES + 256;
// K columns per ring stage (4 chunks of 16 B: 4 TF32 or 8 FP16 each) and per TMEM chain (1024)
template <bool F16> struct Fmt {
  static constexpr int KS = F16 ? 32 : 16, KS_LOG = F16 ? 5 : 4, SUB_STAGES = 1024 / KS;
  static constexpr int SPB = TN / KS;        // stages of a site tile's diagonal block
};
constexpr float Z_SCALE = 8.0f;              // FP16 normals: 2^3 z (|z| < 6.7)
constexpr int L_TOP = 12;                    // FP16 factor: largest |entry| scaled into [2^12, 2^13)
constexpr int LMAX_BLOCKS = 148, SCALE_SLOT = 160, SCALE_FLOATS = 256;
}  // namespace lg

// v = hi + lo in FP16 (round to nearest each): |v - hi - lo| <= 2^-22 |v| while lo is a normal number.
// Two values at a time: cvt.rn.f16x2.f32 (F2FP.PACK_AB) runs on the ALU pipe at full rate; the scalar
// conversion (F2F) shares the quarter-rate unit with the SFU calls of Box-Muller, which bounds the normals.
__device__ __forceinline__ void split_f16x2(float a, float b, uint32_t& hi, uint32_t& lo) {
  const __half2 h = __floats2half2_rn(a, b);
  const float2 f = __half22float2(h);
  const __half2 l = __floats2half2_rn(a - f.x, b - f.y);
  hi = *reinterpret_cast<const uint32_t*>(&h);
  lo = *reinterpret_cast<const uint32_t*>(&l);
}

// 16-byte chunk c of particle i: one Philox quad (TF32) or two (FP16: quads 2c, 2c + 1, scaled by 8),
// split hi / lo.  SFU Box-Muller (philox.cuh, R2).  Quads beyond the lattice (K padding) stay
// zero; sites >= V inside the last quad meet zero columns.
template <bool F16>
__device__ __forceinline__ void normals_chunk(uint64_t seed, uint32_t tag, uint32_t t, int i, int c, int N,
                                              int V, uint4& hi, uint4& lo) {
  if constexpr (F16) {
    // (no branches: several chunks are in flight per thread and their Philox chains must interleave)
    float z[8];
    normals4_fast(seed, tag, t, (uint32_t)i, (uint32_t)(2 * c), z);
    normals4_fast(seed, tag, t, (uint32_t)i, (uint32_t)(2 * c + 1), z + 4);
    const float s0 = (i < N && 8 * c < V) ? lg::Z_SCALE : 0.f, s1 = (i < N && 8 * c + 4 < V) ? lg::Z_SCALE : 0.f;
    split_f16x2(s0 * z[0], s0 * z[1], hi.x, lo.x);
    split_f16x2(s0 * z[2], s0 * z[3], hi.y, lo.y);
    split_f16x2(s1 * z[4], s1 * z[5], hi.z, lo.z);
    split_f16x2(s1 * z[6], s1 * z[7], hi.w, lo.w);
  } else {
    float z[4] = {0.f, 0.f, 0.f, 0.f};
    if (i < N && 4 * c < V) normals4_fast(seed, tag, t, (uint32_t)i, (uint32_t)c, z);
    float h[4];
#pragma unroll
    for (int e = 0; e < 4; ++e) h[e] = tc::tf32_rna(z[e]);
    hi = make_uint4(__float_as_uint(h[0]), __float_as_uint(h[1]), __float_as_uint(h[2]), __float_as_uint(h[3]));
    lo = make_uint4(__float_as_uint(z[0] - h[0]), __float_as_uint(z[1] - h[1]), __float_as_uint(z[2] - h[2]),
                    __float_as_uint(z[3] - h[3]));
  }
}

// z of step t for every particle, hi/lo split, stage-major interleave layout: 16-byte chunk c of
// particle row pr in tile m sits at chunk index (((m * nst + c / 4) * 2 + part) * 4 + c % 4) * 128 + pr,
// part 0 = hi, 1 = lo; a chunk is one Philox quad (TF32) or two (FP16: quads 2c, 2c + 1, scaled by 8).
template <bool F16>
__global__ void __launch_bounds__(128)
normals_split_kernel(uint4* __restrict__ Zs, int N, int ntm, int V, int Kp, int cpb,
                     uint64_t seed, uint32_t tag, uint32_t t, const Ctrl* ctrl, int respect_done) {
  pdl_enter();
  if (respect_done && ctrl->done) return;
  // blockIdx.z: step t + z of a batch, written behind the z steps before it (small populations draw
  // several steps per launch: one step alone is a launch-latency-sized kernel)
  t += blockIdx.z;
  Zs += (size_t)blockIdx.z * ((size_t)ntm * lg::TILE * (size_t)(F16 ? Kp >> 2 : Kp >> 1));
  const int m = blockIdx.x, pr = threadIdx.x;
  const int i = m * lg::TILE + pr, nch = F16 ? Kp >> 3 : Kp >> 2;
  // SFU Box-Muller (philox.cuh, R2).  Quads beyond the lattice (K padding) stay zero;
  // sites >= V inside the last quad meet zero columns.
#pragma unroll 2
  for (int cc = 0; cc < cpb; ++cc) {
    const int c = blockIdx.y * cpb + cc;
    if (c >= nch) break;
    uint4 hi, lo;
    normals_chunk<F16>(seed, tag, t, i, c, N, V, hi, lo);
    const size_t o = ((((size_t)m * (nch >> 2) + (c >> 2)) * 2) * 4 + (c & 3)) * lg::TILE + pr;
    Zs[o] = hi;
    Zs[o + 4 * lg::TILE] = lo;
  }
}

// ---- operand layouts: one bulk copy per operand per stage ------------------------------------
// (Round 1 issued ten copies per stage -- 2 parts of normals, 2 K-steps x 2 chunks x 2 parts of
// s*Lc; the ncu source view showed the producer warp never waiting for a free stage while the
// MMA thread polled "stage full" ~30 times per stage: the copy issue was the bottleneck.)
// Normals: Zs[m][it][part][4 chunks][128 rows][16 B] -- 16 KB per (particle tile, stage).
// s*Lc:    Lt[tn][it][part][kk][c][nrows][16 B], nrows = the rows of site tile tn that K-stage it
//          can reach: 256 below the diagonal block, 256 - KS j in its j-th stage (both K-steps of
//          a stage start at row xs = KS it).  32 nrows floats (128 nrows bytes) per stage; rows
//          above the diagonal are never stored or multiplied.  Offsets below are in 4-byte units.
template <bool F16>
__host__ __device__ inline size_t lt_tile_base(int tn) {          // floats before site tile tn
  using F = lg::Fmt<F16>;
  const size_t diag = (size_t)32 * (256 * F::SPB - F::KS * (F::SPB * (F::SPB - 1) / 2));
  return (size_t)8192 * F::SPB * ((size_t)tn * (tn - 1) / 2) + diag * tn;
}
template <bool F16>
__host__ __device__ inline size_t lt_stage_off(int tn, int it) {  // floats before stage it of tile tn
  using F = lg::Fmt<F16>;
  const int d0 = F::SPB * tn;
  if (it < d0) return lt_tile_base<F16>(tn) + (size_t)it * 8192;
  const int j = it - d0;
  return lt_tile_base<F16>(tn) + (size_t)d0 * 8192 + (size_t)32 * (256 * j - F::KS * (j * (j - 1) / 2));
}

// max |Lc[x][y]|, y <= x, per block (FP16 path: the scale of the factor); no atomics, no reset
__global__ void __launch_bounds__(256) labsmax_kernel(const float* __restrict__ Lc, int V,
                                                      float* __restrict__ blockmax, const Ctrl* ctrl,
                                                      int respect_done) {
  pdl_enter();
  if (respect_done && ctrl->done) return;
  float m = 0.f;
  for (int x = blockIdx.x; x < V; x += gridDim.x)
    for (int y = threadIdx.x; y <= x; y += blockDim.x) m = fmaxf(m, fabsf(Lc[(size_t)x * V + y]));
  __shared__ float red[8];
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) m = fmaxf(m, __shfl_xor_sync(0xffffffffu, m, o));
  if ((threadIdx.x & 31) == 0) red[threadIdx.x >> 5] = m;
  __syncthreads();
  if (threadIdx.x == 0) {
    for (int w = 1; w < 8; ++w) m = fmaxf(m, red[w]);
    blockmax[blockIdx.x] = m;
  }
}

// c = 2^(L_TOP - floor(log2(s max|Lc|))): the largest scaled entry lies in [2^12, 2^13)
__device__ inline float l_scale_of(const float* blockmax, float s) {
  float m = 0.f;
  for (int b = threadIdx.x & 31; b < lg::LMAX_BLOCKS; b += 32) m = fmaxf(m, blockmax[b]);
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) m = fmaxf(m, __shfl_xor_sync(0xffffffffu, m, o));
  m *= fabsf(s);
  if (!(m > 0.f) || !isfinite(m)) return 1.f;
  return ldexpf(1.f, lg::L_TOP - ilogbf(m));
}

// one thread per (row x, 16-byte chunk of columns): TF32 4 columns, FP16 8
template <bool F16>
__global__ void lsplit_tiled_kernel(const float* __restrict__ Lc, int V, int Vn, int Kp, float s,
                                    float* __restrict__ out, float* __restrict__ scale,
                                    const Ctrl* ctrl, int respect_done) {
  pdl_enter();
  if (respect_done && ctrl->done) return;
  using F = lg::Fmt<F16>;
  constexpr int CW = F16 ? 8 : 4;                      // columns per chunk
  float c = 1.f;
  if constexpr (F16) {
    c = l_scale_of(scale, s);
    // the GEMM epilogue undoes both scales: exact powers of two
    if (blockIdx.x == 0 && threadIdx.x == 0) scale[lg::SCALE_SLOT] = 1.0f / (c * lg::Z_SCALE);
  }
  const size_t idx = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (idx >= (size_t)(Kp / CW) * Vn) return;
  const int yc = (int)(idx / Vn), x = (int)(idx - (size_t)yc * Vn), y0 = yc * CW;
  const int tn = x >> 8, n0 = tn << 8, it = y0 >> F::KS_LOG;
  const int rs = max(n0, F::KS * it);
  if (x < rs) return;                                // above the diagonal: never multiplied
  const int nrows = n0 + 256 - rs;
  const int kc = (y0 & (F::KS - 1)) / CW;            // chunk of the stage: kk = kc / 2, c = kc % 2
  float v[CW];
#pragma unroll
  for (int e = 0; e < CW; ++e) {
    const int y = y0 + e;
    v[e] = (x < V && y < V && y <= x) ? c * s * Lc[(size_t)x * V + y] : 0.f;
  }
  uint4 hi, lo;
  if constexpr (F16) {
    split_f16x2(v[0], v[1], hi.x, lo.x);
    split_f16x2(v[2], v[3], hi.y, lo.y);
    split_f16x2(v[4], v[5], hi.z, lo.z);
    split_f16x2(v[6], v[7], hi.w, lo.w);
  } else {
    float h[4];
#pragma unroll
    for (int e = 0; e < 4; ++e) h[e] = tc::tf32_rna(v[e]);
    hi = make_uint4(__float_as_uint(h[0]), __float_as_uint(h[1]), __float_as_uint(h[2]), __float_as_uint(h[3]));
    lo = make_uint4(__float_as_uint(tc::tf32_rna(v[0] - h[0])), __float_as_uint(tc::tf32_rna(v[1] - h[1])),
                    __float_as_uint(tc::tf32_rna(v[2] - h[2])), __float_as_uint(tc::tf32_rna(v[3] - h[3])));
  }
  uint4* o = reinterpret_cast<uint4*>(out + lt_stage_off<F16>(tn, it)) + (size_t)kc * nrows + (x - rs);
  o[0] = hi;
  o[(size_t)4 * nrows] = lo;                         // part stride: 2 kk x 2 c x nrows chunks
}

struct ProposeTcParams {
  const float* phi; float* phip;     // [V][ld]
  const float* Zs;                   // normals_split_kernel output
  const float* Lsplit;               // s*Lc hi | lo per (site tile, K-stage): lt_stage_off
  const float* scale_inv;            // FP16 operands: 1 / (factor scale x normal scale), else unused
  // normals of the NEXT step, drawn by warps 10-11 of every CTA while the tensor core works
  // (nullptr: none).  A separate kernel cannot do this: beside a GEMM CTA no register file has room
  // for another block, so its blocks only start once GEMM CTAs exit (CUPTI timeline).
  uint4* Znext;
  int N;
  uint64_t seed;
  uint32_t tag, t_next;
  const Ctrl* ctrl;
  int ld, V, Vn, Kp, ntm, ntn;       // Vn = V rounded up to 256 rows, Kp = V rounded up to a K-stage
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

template <bool F16>
__global__ void __launch_bounds__(lg::THREADS, 1) propose_tc_kernel(const ProposeTcParams p) {
  using namespace tc;
  using namespace lg;
  using F = Fmt<F16>;
  constexpr int KS = F::KS, SUB_STAGES = F::SUB_STAGES;
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

  if (warp >= 8) {
  asm volatile("setmaxnreg.dec.sync.aligned.u32 %0;" ::"n"(REGS_REST));
  if (warp == 8) {
    // ================================ producer: two bulk copies per stage =====================
    if (lane == 0) {
      int s = 0;
      uint32_t ph = 0;
      const int nstz = Kp >> F::KS_LOG;
      // s*Lc blocks are re-read by every particle tile for the whole launch: evict_last.  The normals of
      // a particle tile are dead after one work item; with the same hint they crowded the factor out.
      const uint64_t keep = l2_policy_evict_last();
      for (TileIter ti(p.ntm, p.ntn, p.pair); ti.valid(); ti.next()) {
        int m, tn;
        ti.tile(m, tn);
        const int n0 = tn * TN;
        const int nst = min(n0 + TN, Kp) >> F::KS_LOG;       // K-stages up to the tile's last row
        const float* za = p.Zs + (size_t)m * nstz * (2 * A_PART / 4);
        for (int it = 0; it < nst; ++it) {
          const uint32_t st = ring + (uint32_t)s * STAGE_BYTES;
          const int nrows = n0 + TN - max(n0, KS * it);      // rows of the s*Lc block of this stage
          const uint32_t bbytes = 128u * (uint32_t)nrows;    // 2 parts x 2 kk x 2 c x nrows x 16 B
          mbar_wait(empty(s), ph ^ 1);
          mbar_expect_tx(full(s), 2 * A_PART + bbytes);
          bulk_g2s(st, za + (size_t)it * (2 * A_PART / 4), 2 * A_PART, full(s));
          bulk_g2s_hint(st + 2 * A_PART, p.Lsplit + lt_stage_off<F16>(tn, it), bbytes, full(s), keep);
          if (++s == STAGES) { s = 0; ph ^= 1; }
        }
      }
    }
    __syncwarp();
  } else if (warp >= GEN_WARP0) {
    // ================================ normals of the next step ================================
    if (p.Znext) {
      const int nch = F16 ? Kp >> 3 : Kp >> 2;             // 16-byte chunks per particle row
      // flat index over (particle tile, chunk, particle row): consecutive threads, consecutive rows
      const long long total = (long long)p.ntm * nch * TILE;
      const long long stride = (long long)gridDim.x * GEN_THREADS;
      for (long long idx = (long long)blockIdx.x * GEN_THREADS + (threadIdx.x - GEN_WARP0 * 32); idx < total;
           idx += stride) {
        const int pr = (int)(idx & (TILE - 1)), mc = (int)(idx >> 7);
        const int m = mc / nch, c = mc - m * nch, i = m * TILE + pr;
        uint4 hi, lo;
        normals_chunk<F16>(p.seed, p.tag, p.t_next, i, c, p.N, V, hi, lo);
        const size_t o = ((((size_t)m * (nch >> 2) + (c >> 2)) * 2) * 4 + (c & 3)) * TILE + pr;
        p.Znext[o] = hi;
        p.Znext[o + 4 * TILE] = lo;
      }
    }
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
        const int nst = min(n0 + TN, Kp) >> F::KS_LOG;
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
            // both K-steps of a stage reach the same rows (xs = KS it); the block sits packed in
            // the stage as [part][kk][c][nrows][16 B], so LBO and the part stride follow nrows
            const int rowstart = max(n0, KS * it), nrows = n0 + TN - rowstart;
            const uint32_t idesc = F16 ? instr_desc_f16(TILE, nrows) : instr_desc(TILE, nrows);
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
              // (n0 is a multiple of 256 <= KS it0 whenever it0 > 0), so no column is left stale.
              if constexpr (F16) {
                tc_mma_f16(d, a_lo, b_hi, idesc, (it != it0) || kk);
                tc_mma_f16(d, a_hi, b_lo, idesc, 1);
                tc_mma_f16(d, a_hi, b_hi, idesc, 1);
              } else {
                tc_mma_tf32(d, a_lo, b_hi, idesc, (it != it0) || kk);
                tc_mma_tf32(d, a_hi, b_lo, idesc, 1);
                tc_mma_tf32(d, a_hi, b_hi, idesc, 1);
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
  }
  } else {
    asm volatile("setmaxnreg.inc.sync.aligned.u32 %0;" ::"n"(REGS_EPI));
    // ================================ epilogue: phi' = phi + sum of chains ====================
    // warp w: TMEM lane quarter w % 4 (32 particles), column half w / 4 (128 sites)
    int cnt = 0;
    const int Q = warp & 3, hc = warp >> 2;
    const uint32_t tlane = taddr + ((uint32_t)(Q * 32) << 16);
    const float inv = F16 ? __ldg(p.scale_inv) : 1.f;   // (exact power of two)
    for (TileIter ti(p.ntm, p.ntn, p.pair); ti.valid(); ti.next()) {
      int m, tn;
      ti.tile(m, tn);
      const int n0 = tn * TN;
      const int nst = min(n0 + TN, Kp) >> F::KS_LOG;
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
          f[j] = (x0 + j < V) ? __ldcs(p.phi + (size_t)(x0 + j) * p.ld + col) : 0.f;
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
              p.phip[(size_t)(x0 + cb + jj) * p.ld + col] = fmaf(__uint_as_float(r0[jj]), inv, f[cb + jj]);
#pragma unroll
          for (int jj = 0; jj < 16; ++jj)
            if (x0 + cb + 16 + jj < V)
              p.phip[(size_t)(x0 + cb + 16 + jj) * p.ld + col] = fmaf(__uint_as_float(r1[jj]), inv, f[cb + 16 + jj]);
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
            f[jj] = (x0 + cb + jj < V) ? __ldcs(p.phi + (size_t)(x0 + cb + jj) * p.ld + col) : 0.f;
#pragma unroll
          for (int jj = 0; jj < 16; ++jj)
            if (x0 + cb + jj < V) p.phip[(size_t)(x0 + cb + jj) * p.ld + col] = fmaf(acc[cb + jj], inv, f[jj]);
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

// s*Lc split hi / lo in the tiled layout propose_tc_kernel streams (lt_stage_off); the FP16 form
// keeps its per-block maxima and the inverse scale in the SCALE_FLOATS floats behind the operand
static float* scale_of(float* Lsplit, int V) {
  return Lsplit + lt_tile_base<true>(round_up(V, lg::TN) / lg::TN);
}

void launch_propose_lsplit(const float* Lc, int V, int ld, float s, float* Lsplit, const Ctrl* ctrl,
                           int respect_done, cudaStream_t st, bool f16) {
  (void)ld;
  int Vn, Kp;
  propose_tc_dims(V, &Vn, &Kp, f16);
  if (f16) {
    ++g_launches;
    launch_pdl(labsmax_kernel, lg::LMAX_BLOCKS, 256, 0, st, Lc, V, scale_of(Lsplit, V), ctrl, respect_done);
    ++g_launches;
    launch_pdl(lsplit_tiled_kernel<true>, (unsigned)(((size_t)(Kp / 8) * Vn + 255) / 256), 256, 0, st, Lc, V,
               Vn, Kp, s, Lsplit, scale_of(Lsplit, V), ctrl, respect_done);
  } else {
    ++g_launches;
    launch_pdl(lsplit_tiled_kernel<false>, (unsigned)(((size_t)(Kp / 4) * Vn + 255) / 256), 256, 0, st, Lc, V,
               Vn, Kp, s, Lsplit, (float*)nullptr, ctrl, respect_done);
  }
}

void propose_tc_dims(int V, int* Vn, int* Kp, bool f16) {
  *Vn = round_up(V, lg::TN);
  *Kp = round_up(V, f16 ? 32 : 16);
}

// floats of the split normals of ONE step
size_t propose_tc_zstep_floats(int V, int ld, bool f16) {
  return f16 ? (size_t)round_up(V, 32) * ld : (size_t)2 * round_up(V, 16) * ld;
}
// steps of normals drawn per launch: small populations (whose GEMM cannot hide the next step's normals)
// draw a batch, FP16 only
int propose_tc_zbatch(int V, int ld, bool f16) {
  return (f16 && (size_t)ld * V < ((size_t)1 << 22)) ? 8 : 1;
}
// (sized for either format: one TF32 step or the FP16 batch)
size_t propose_tc_zsplit_floats(int V, int ld) {
  const size_t a = propose_tc_zstep_floats(V, ld, false);
  const size_t b = propose_tc_zstep_floats(V, ld, true) * propose_tc_zbatch(V, ld, true);
  return a > b ? a : b;
}

size_t propose_tc_lsplit_floats(int V) {
  const int ntn = round_up(V, lg::TN) / lg::TN;
  const size_t a = lt_tile_base<false>(ntn), b = lt_tile_base<true>(ntn) + lg::SCALE_FLOATS;
  return a > b ? a : b;
}

void launch_normals_split(float* Zs, int N, int ld, int V, uint64_t seed, uint32_t tag, uint32_t t,
                          const Ctrl* ctrl, int respect_done, cudaStream_t st, bool f16, int nsteps) {
  const int Kp = round_up(V, f16 ? 32 : 16);
  const int nch = f16 ? Kp / 8 : Kp / 4;             // 16-byte chunks per particle row
  // chunks per thread: one per block made 1 M blocks at C4 (block-launch-rate bound); a small
  // population keeps one per thread so that the grid still fills the GPU
  int cpb = (ld / lg::TILE) * nch * nsteps / (148 * 16);
  const int cmax = f16 ? 4 : 8;
  cpb = cpb < 1 ? 1 : cpb > cmax ? cmax : cpb;
  dim3 grid(ld / lg::TILE, (nch + cpb - 1) / cpb, nsteps);
  ++g_launches;
  if (f16)
    launch_pdl(normals_split_kernel<true>, grid, 128, 0, st, reinterpret_cast<uint4*>(Zs), N, ld / lg::TILE, V,
               Kp, cpb, seed, tag, t, ctrl, respect_done);
  else
    launch_pdl(normals_split_kernel<false>, grid, 128, 0, st, reinterpret_cast<uint4*>(Zs), N, ld / lg::TILE, V,
               Kp, cpb, seed, tag, t, ctrl, respect_done);
}

void launch_propose_tc(const float* phi, float* phip, const float* Zs, const float* Lsplit, int ld,
                       int V, const Ctrl* ctrl, int respect_done, cudaStream_t st, bool f16,
                       const NextNormals* next) {
  static bool attr_done = false;
  if (!attr_done) {
    cudaFuncSetAttribute(propose_tc_kernel<false>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                         lg::SMEM_BYTES);
    cudaFuncSetAttribute(propose_tc_kernel<true>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                         lg::SMEM_BYTES);
    attr_done = true;
  }
  const int num_sms = num_sms_cached();
  ProposeTcParams p;
  p.phi = phi; p.phip = phip; p.Zs = Zs; p.Lsplit = Lsplit; p.ctrl = ctrl;
  p.scale_inv = f16 ? scale_of(const_cast<float*>(Lsplit), V) + lg::SCALE_SLOT : nullptr;
  p.Znext = next ? reinterpret_cast<uint4*>(next->Zs) : nullptr;
  p.N = next ? next->N : 0; p.seed = next ? next->seed : 0; p.tag = next ? next->tag : 0;
  p.t_next = next ? next->t : 0;
  p.ld = ld; p.V = V;
  propose_tc_dims(V, &p.Vn, &p.Kp, f16);
  p.ntm = ld / lg::TILE; p.ntn = p.Vn / lg::TN; p.respect_done = respect_done;
  p.pair = p.ntm * p.ntn > num_sms;
  const int nunits = p.ntm * (p.pair ? (p.ntn + 1) / 2 : p.ntn);
  const int grid = nunits < num_sms ? nunits : num_sms;
  ++g_launches;
  if (f16) launch_pdl(propose_tc_kernel<true>, grid, lg::THREADS, lg::SMEM_BYTES, st, p);
  else launch_pdl(propose_tc_kernel<false>, grid, lg::THREADS, lg::SMEM_BYTES, st, p);
}

}  // namespace phi4
