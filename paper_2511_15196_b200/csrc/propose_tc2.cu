// propose_tc2.cu -- the large-V proposal GEMM of propose_tc.cu on CTA pairs (tcgen05
// cta_group::2): phi'[x][i] = phi[x][i] + sum_{y<=x} (s Lc)[x][y] z[y][i] in 3xTF32
// (BASELINE.json north_star; PAPER.md:53(i), :172).
//
// Why pairs.  The one-CTA kernel streams 48 KB of operands per K = 16 stage (16 KB of normals, 32 KB
// of s*Lc) for 768 tensor cycles: 62 B/clk per SM, 12 TB/s over the chip at C4 -- the measured
// L2 -> SM throughput of the part (ncu: lts 12.3 TB/s, tensor pipe 80 %).  It is bound by the L2
// fabric, not by the tensor pipe.  A CTA pair computes a 256-particle x 256-site tile with one
// M = 256 instruction: each CTA keeps its own 128 particles of normals and only HALF of the
// s*Lc rows (the hardware reads the other half from the peer's shared memory), so a stage is
// 32 KB per SM: a third less L2 traffic for the same flops, and six ring stages instead of four.
//
// Roles per CTA (320 threads): warps 0-7 epilogue (tcgen05.ld of the CTA's own 128 TMEM lanes,
// phi' = phi + d), warp 8 bulk-copy producer (own normals, own half of the s*Lc block), warp 9:
// in the leader (cluster rank 0) the MMA issuer, in the peer a relay that forwards "my stage is
// full" to the leader's barrier.  tcgen05.commit multicasts "stage free" / "accumulator full" to
// both CTAs; the peer's epilogue warps arrive on the leader's "accumulator drained" barrier.
// Tile order, accumulation chains (K = 1024 per TMEM chain) and operand layouts are those of
// propose_tc.cu; used when the padded population is a multiple of 256 and fills the GPU.
#include <cstdlib>

#include "kernels.cuh"
#include "tcgen05.cuh"

namespace phi4 {

namespace lg2 {
constexpr int TILE = 128;                    // particles per CTA = TMEM lanes
constexpr int TN = 256;                      // sites per output tile = TMEM columns per buffer
constexpr int HN = TN / 2;                   // rows of s*Lc held by one CTA
constexpr int STAGES = 6;
constexpr int CHUNK_A = TILE * 16;           // one 16-byte K-chunk of 128 rows
constexpr int CHUNK_B = HN * 16;
constexpr int A_PART = 4 * CHUNK_A;          // K = 16 per stage: 4 chunks per hi / lo part
constexpr int B_PART = 4 * CHUNK_B;
constexpr int STAGE_BYTES = 2 * A_PART + 2 * B_PART;   // 32 KB
constexpr int THREADS = 320;
constexpr int SUB_STAGES = 64;               // one TMEM accumulation chain covers K = 1024
constexpr int SMEM_BYTES = STAGES * STAGE_BYTES + 256;
}  // namespace lg2

namespace tc {
__device__ __forceinline__ uint32_t cluster_ctarank() {
  uint32_t r;
  asm volatile("mov.u32 %0, %%cluster_ctarank;" : "=r"(r));
  return r;
}
__device__ __forceinline__ void cluster_sync_all() {
  asm volatile("barrier.cluster.arrive.release.aligned;" ::: "memory");
  asm volatile("barrier.cluster.wait.acquire.aligned;" ::: "memory");
}
// arrive on the barrier at the same shared-memory offset in CTA `rank` of the cluster
__device__ __forceinline__ void mbar_arrive_remote(uint32_t bar, uint32_t rank) {
  asm volatile(
      "{\n\t"
      ".reg .b32 ra;\n\t"
      "mapa.shared::cluster.u32 ra, %0, %1;\n\t"
      "mbarrier.arrive.release.cluster.shared::cluster.b64 _, [ra];\n\t"
      "}" ::"r"(bar), "r"(rank)
      : "memory");
}
__device__ __forceinline__ void mbar_wait_cluster(uint32_t bar, uint32_t parity) {
  asm volatile(
      "{\n\t"
      ".reg .pred p;\n\t"
      "WAITC_%=:\n\t"
      "mbarrier.try_wait.parity.acquire.cluster.shared::cta.b64 p, [%0], %1;\n\t"
      "@p bra DONEC_%=;\n\t"
      "bra WAITC_%=;\n\t"
      "DONEC_%=:\n\t"
      "}" ::"r"(bar), "r"(parity)
      : "memory");
}
__device__ __forceinline__ void tmem_alloc2(uint32_t slot, uint32_t ncols) {
  asm volatile("tcgen05.alloc.cta_group::2.sync.aligned.shared::cta.b32 [%0], %1;" ::"r"(slot),
               "r"(ncols)
               : "memory");
  asm volatile("tcgen05.relinquish_alloc_permit.cta_group::2.sync.aligned;" ::: "memory");
}
__device__ __forceinline__ void tmem_dealloc2(uint32_t taddr, uint32_t ncols) {
  asm volatile("tcgen05.dealloc.cta_group::2.sync.aligned.b32 %0, %1;" ::"r"(taddr), "r"(ncols)
               : "memory");
}
// completion of all earlier MMAs of this thread arrives on `bar` in both CTAs of the pair
__device__ __forceinline__ void tc_commit2(uint32_t bar) {
  asm volatile(
      "tcgen05.commit.cta_group::2.mbarrier::arrive::one.shared::cluster.multicast::cluster.b64 "
      "[%0], %1;" ::"r"(bar),
      "h"((uint16_t)3)
      : "memory");
}
// D[tmem, 256 rows over the pair] (+)= A[smem, 128 rows per CTA] * B[smem, N/2 rows per CTA]^T
__device__ __forceinline__ void tc_mma2_tf32(uint32_t d, uint64_t a, uint64_t b, uint32_t idesc,
                                             uint32_t accumulate) {
  asm volatile(
      "{\n\t"
      ".reg .pred p;\n\t"
      "setp.ne.b32 p, %4, 0;\n\t"
      "tcgen05.mma.cta_group::2.kind::tf32 [%0], %1, %2, %3, p;\n\t"
      "}" ::"r"(d), "l"(a), "l"(b), "r"(idesc), "r"(accumulate)
      : "memory");
}
}  // namespace tc

// ---- operand layouts of the pair kernel: one bulk copy per operand per stage -----------------
// (ten copies per stage -- 2 parts of normals, 2 K-steps x 2 chunks x 2 parts of s*Lc -- kept the
// producer warp busy for ~1500 cycles per 768-cycle stage: ncu source view, round 1.)
// Normals: Zs[m][it][part][4 chunks][128 rows][4] -- 16 KB per (particle tile, stage).
// s*Lc:    Lt[tn][it][rank][part][kk][c][hr rows][4], hr = half of the rows of site tile tn that
//          K-stage it can reach (256 below the diagonal block, 256 - 16 j in its j-th stage):
//          32 nrows floats per stage, each CTA's half contiguous.
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
  const int hr = (n0 + 256 - rs) >> 1;
  const int r = (x - rs) / hr, row = (x - rs) - r * hr;
  const int kk = (y >> 3) & 1, c = (y >> 2) & 1, e = y & 3;
  const float v = (x < V && y < V && y <= x) ? s * Lc[(size_t)x * V + y] : 0.f;
  const float hi = tc::tf32_rna(v), lo = tc::tf32_rna(v - hi);
  const size_t o = lt_stage_off(tn, it) + (size_t)r * 32 * hr +
                   ((size_t)((kk * 2 + c) * hr + row)) * 4 + e;
  out[o] = hi;
  out[o + (size_t)16 * hr] = lo;                     // part stride: 2 kk x 2 c x hr rows x 4
}

struct ProposeTc2Params {
  const float* phi; float* phip;     // [V][ld]
  const float* Zs;                   // normals_split_kernel output
  const float* Lsplit;               // packed s*Lc hi | lo (tcgen05.cuh layout)
  const Ctrl* ctrl;
  int ld, V, Vn, Kp, ntm, ntn;       // Vn = V rounded up to 256 rows, Kp = V rounded up to 16
  int respect_done;
};

// Work items of a cluster: (pair of particle tiles mp, pair of site tiles (j, ntn-1-j)); see
// TileIter in propose_tc.cu -- every item spans ntn+1 K-blocks of 256, clusters stay in step and
// the clusters that hold the same particle tiles stream the same normals through L2 together.
struct Tile2Iter {
  int np, nunits, ntn, u, half, stride;
  __device__ Tile2Iter(int ntm, int ntn_)
      : np((ntn_ + 1) >> 1), nunits((ntm >> 1) * ((ntn_ + 1) >> 1)), ntn(ntn_),
        u(blockIdx.x >> 1), half(0), stride(gridDim.x >> 1) {}
  __device__ bool valid() const { return u < nunits; }
  __device__ void tile(int& mp, int& n) const {
    mp = u / np;
    const int j = u % np;
    n = half ? ntn - 1 - j : j;
  }
  __device__ void next() {
    const int j = u % np;
    if (!half && ntn - 1 - j != j) { half = 1; return; }
    half = 0;
    u += stride;
  }
};

__global__ void __cluster_dims__(2, 1, 1) __launch_bounds__(lg2::THREADS, 1)
propose_tc2_kernel(const ProposeTc2Params p) {
  using namespace tc;
  using namespace lg2;
  extern __shared__ __align__(1024) uint8_t smem[];
  pdl_trigger();
  uint64_t* bars = reinterpret_cast<uint64_t*>(smem + STAGES * STAGE_BYTES);
  const uint32_t bar0 = smem_u32(bars);
  auto full = [&](int s) { return bar0 + 8u * s; };
  auto empty = [&](int s) { return bar0 + 8u * (STAGES + s); };
  auto pfull = [&](int s) { return bar0 + 8u * (2 * STAGES + s); };        // leader: peer's stage is full
  auto dfull = [&](int b) { return bar0 + 8u * (3 * STAGES + b); };
  auto dempty = [&](int b) { return bar0 + 8u * (3 * STAGES + 2 + b); };   // leader: 16 epilogue warps
  uint32_t* tmem_slot = reinterpret_cast<uint32_t*>(bars + 3 * STAGES + 4);
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const uint32_t rank = cluster_ctarank();
  const int V = p.V, Vn = p.Vn, Kp = p.Kp, nkc = Kp >> 2; (void)nkc;

  if (warp == 8 && lane == 0) {
    for (int s = 0; s < STAGES; ++s) { mbar_init(full(s), 1); mbar_init(empty(s), 1); mbar_init(pfull(s), 1); }
    for (int b = 0; b < 2; ++b) { mbar_init(dfull(b), 1); mbar_init(dempty(b), 16); }
    fence_mbar_init();
  }
  if (warp == 0) tmem_alloc2(smem_u32(tmem_slot), 2 * TN);
  tc_fence_before();
  cluster_sync_all();                 // barriers of both CTAs initialised, TMEM allocated in both
  tc_fence_after();
  const uint32_t taddr = *tmem_slot;
  const uint32_t ring = smem_u32(smem);
  pdl_wait();
  const bool skip = p.respect_done && p.ctrl->done;

  if (skip) {
    // nothing was issued: fall through to the common teardown
  } else if (warp == 8) {
    // ================================ producer: two bulk copies per stage =====================
    if (lane == 0) {
      int s = 0;
      uint32_t ph = 0;
      const int nstz = Kp >> 4;
      for (Tile2Iter ti(p.ntm, p.ntn); ti.valid(); ti.next()) {
        int mp, tn;
        ti.tile(mp, tn);
        const int m = 2 * mp + (int)rank, n0 = tn * TN;
        const int nst = min(n0 + TN, Kp) >> 4;               // K-stages up to the tile's last row
        const float* za = p.Zs + (size_t)m * nstz * (2 * A_PART / 4);
        for (int it = 0; it < nst; ++it) {
          const uint32_t st = ring + (uint32_t)s * STAGE_BYTES;
          const int hr = (n0 + TN - max(n0, 16 * it)) >> 1;  // this CTA's rows of the s*Lc block
          const uint32_t bbytes = 128u * (uint32_t)hr;       // 2 parts x 2 kk x 2 c x hr x 16 B
          mbar_wait(empty(s), ph ^ 1);
          mbar_expect_tx(full(s), 2 * A_PART + bbytes);
          bulk_g2s(st, za + (size_t)it * (2 * A_PART / 4), 2 * A_PART, full(s));
          bulk_g2s(st + 2 * A_PART, p.Lsplit + lt_stage_off(tn, it) + (size_t)rank * 32 * hr, bbytes,
                   full(s));
          if (++s == STAGES) { s = 0; ph ^= 1; }
        }
      }
    }
    __syncwarp();
  } else if (warp == 9) {
    if (lane == 0 && rank != 0) {
      // ================================ peer: relay "stage full" to the leader ================
      int s = 0;
      uint32_t ph = 0;
      for (Tile2Iter ti(p.ntm, p.ntn); ti.valid(); ti.next()) {
        int mp, tn;
        ti.tile(mp, tn);
        const int nst = min(tn * TN + TN, Kp) >> 4;
        for (int it = 0; it < nst; ++it) {
          mbar_wait(full(s), ph);
          mbar_arrive_remote(pfull(s), 0);
          if (++s == STAGES) { s = 0; ph ^= 1; }
        }
      }
    } else if (lane == 0) {
      // ================================ leader: MMA issuer =====================================
      int s = 0, cnt = 0;
      uint32_t ph = 0;
      const uint64_t a_base = smem_desc(ring, CHUNK_A, 128);
      for (Tile2Iter ti(p.ntm, p.ntn); ti.valid(); ti.next()) {
        int mp, tn;
        ti.tile(mp, tn);
        const int n0 = tn * TN;
        const int nst = min(n0 + TN, Kp) >> 4;
        for (int it0 = 0; it0 < nst; it0 += SUB_STAGES, ++cnt) {
          const int buf = cnt & 1;
          mbar_wait_cluster(dempty(buf), ((cnt >> 1) & 1) ^ 1);
          tc_fence_after();
          const uint32_t dbase = taddr + (uint32_t)(buf * TN);
          const int it1 = min(nst, it0 + SUB_STAGES);
          for (int it = it0; it < it1; ++it) {
            mbar_wait(full(s), ph);
            mbar_wait_cluster(pfull(s), ph);
            tc_fence_after();
            const uint32_t so = (uint32_t)s * (STAGE_BYTES >> 4);
            // both K-steps of a stage reach the same rows (xs = 16 it); the block sits packed in
            // the stage: [part][kk][c][hr rows][16 B], so LBO and the part stride follow hr
            const int rowstart = max(n0, 16 * it), nrows = n0 + TN - rowstart, hr = nrows >> 1;
            const uint32_t idesc = instr_desc(2 * TILE, nrows);
            const uint32_t d = dbase + (uint32_t)(rowstart - n0);
            const uint64_t b_st = smem_desc(ring + 2 * A_PART, (uint32_t)hr * 16u, 128) + so;
#pragma unroll
            for (int kk = 0; kk < 2; ++kk) {
              const uint64_t a_hi = a_base + so + (uint32_t)(2 * kk) * (CHUNK_A >> 4);
              const uint64_t a_lo = a_hi + (A_PART >> 4);
              const uint64_t b_hi = b_st + (uint32_t)(2 * kk * hr);
              const uint64_t b_lo = b_hi + (uint32_t)(4 * hr);
              // first K-step of a chain overwrites; see propose_tc.cu for why no column is stale
              tc_mma2_tf32(d, a_lo, b_hi, idesc, (it != it0) || kk);
              tc_mma2_tf32(d, a_hi, b_lo, idesc, 1);
              tc_mma2_tf32(d, a_hi, b_hi, idesc, 1);
            }
            tc_commit2(empty(s));
            if (++s == STAGES) { s = 0; ph ^= 1; }
          }
          tc_commit2(dfull(buf));
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
    auto drained = [&](int buf) {
      tc_fence_before();
      __syncwarp();
      if (lane == 0) {
        if (rank == 0) mbar_arrive(dempty(buf));
        else mbar_arrive_remote(dempty(buf), 0);
      }
    };
    for (Tile2Iter ti(p.ntm, p.ntn); ti.valid(); ti.next()) {
      int mp, tn;
      ti.tile(mp, tn);
      const int m = 2 * mp + (int)rank, n0 = tn * TN;
      const int nst = min(n0 + TN, Kp) >> 4;
      const size_t col = (size_t)m * TILE + Q * 32 + lane;
      const int x0 = n0 + hc * 128;
      if (nst <= SUB_STAGES) {
        const int buf = cnt & 1;
        mbar_wait_relaxed(dfull(buf), (cnt >> 1) & 1);
        tc_fence_after();
        for (int cb = 0; cb < 128; cb += 16) {
          uint32_t r[16];
          tmem_ld16(tlane + (uint32_t)(buf * TN + hc * 128 + cb), r);
          float f[16];
#pragma unroll
          for (int jj = 0; jj < 16; ++jj)
            f[jj] = (x0 + cb + jj < V) ? p.phi[(size_t)(x0 + cb + jj) * p.ld + col] : 0.f;
          tmem_ld_wait();
#pragma unroll
          for (int jj = 0; jj < 16; ++jj)
            if (x0 + cb + jj < V)
              p.phip[(size_t)(x0 + cb + jj) * p.ld + col] = f[jj] + __uint_as_float(r[jj]);
        }
        drained(buf);
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
          drained(buf);
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
  // the peer's shared memory and barriers are in use until the leader's last MMA has completed:
  // both CTAs leave together
  tc_fence_before();
  cluster_sync_all();
  if (warp == 0) tmem_dealloc2(taddr, 2 * TN);
}

// CTA pairs need an even number of particle tiles and enough work to fill every SM pair.
bool propose_tc2_usable(int V, int ld, int num_sms) {
  static const bool on = [] { const char* e = getenv("PHI4_2CTA"); return e && e[0] == '1'; }();
  if (!on || !propose_tc_supported(V) || ld % (2 * lg2::TILE) != 0) return false;
  const int ntn = round_up(V, lg2::TN) / lg2::TN;
  return (ld / (2 * lg2::TILE)) * ((ntn + 1) / 2) >= num_sms / 2;
}

size_t propose_tc2_lsplit_floats(int V) { return lt_tile_base(round_up(V, lg2::TN) / lg2::TN); }

void launch_lsplit_tiled(const float* Lc, int V, float s, float* Lsplit, const Ctrl* ctrl,
                         int respect_done, cudaStream_t st) {
  int Vn, Kp;
  propose_tc_dims(V, &Vn, &Kp);
  ++g_launches;
  launch_pdl(lsplit_tiled_kernel, (unsigned)(((size_t)Kp * Vn + 255) / 256), 256, 0, st, Lc, V, Vn,
             Kp, s, Lsplit, ctrl, respect_done);
}

void launch_propose_tc2(const float* phi, float* phip, const float* Zs, const float* Lsplit,
                        int ld, int V, const Ctrl* ctrl, int respect_done, int num_sms,
                        cudaStream_t st) {
  static bool attr_done = false;
  if (!attr_done) {
    cudaFuncSetAttribute(propose_tc2_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize,
                         lg2::SMEM_BYTES);
    attr_done = true;
  }
  ProposeTc2Params p;
  p.phi = phi; p.phip = phip; p.Zs = Zs; p.Lsplit = Lsplit; p.ctrl = ctrl;
  p.ld = ld; p.V = V;
  propose_tc_dims(V, &p.Vn, &p.Kp);
  p.ntm = ld / lg2::TILE; p.ntn = p.Vn / lg2::TN; p.respect_done = respect_done;
  ++g_launches;
  launch_pdl(propose_tc2_kernel, num_sms & ~1, lg2::THREADS, lg2::SMEM_BYTES, st, p);
}

}  // namespace phi4
