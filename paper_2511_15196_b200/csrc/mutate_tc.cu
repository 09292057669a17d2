// mutate_tc.cu -- M1-M4 fused over the k steps of one temperature on tcgen05 tensor cores.
//
// One CTA owns a tile of 128 particles for all k steps; phi is read from HBM once and written
// once per temperature.  Per step, with D[p, x] = sum_y Z[p, y] * (s Lc)[x, y]:
//   producer warps   Philox normals z (never touch HBM), split hi/lo for 3xTF32, written to a
//                    shared-memory ring in the UMMA K-major "interleave" layout: a Philox quad
//                    (sites 4q..4q+3) is exactly one 16-byte core-matrix row, so a warp stores
//                    512 contiguous bytes
//   MMA thread       tcgen05.mma.kind::tf32, M = 128 particles (TMEM lanes), N = sites (TMEM
//                    columns), K = 8 per instruction; three products per K-step
//                    (z_lo L_hi + z_hi L_lo + z_hi L_hi) into one FP32 TMEM accumulator; rows
//                    x < 8 ks of a K-step are zero (Lc is lower-triangular) and are skipped
//   epilogue warps   tcgen05.ld: thread p owns particle p; phi' = phi + d into the particle's
//                    second shared-memory tile, per-site action differences, Metropolis / hard
//                    constraint accept, commit by flipping the particle's tile pointer
// The accumulator is double-buffered in TMEM so that the MMAs of step t+1 overlap the stencil of
// step t; normals do not depend on the state, so producers run ahead through the ring.
//
// PAPER.md:53(i), :172 (covariance-scaled RW proposal), :29 (Eq. 1), :43 (U0, p_beta);
// BASELINE.json north_star (3xTF32 tcgen05 proposal product, tile kept on-chip across k steps).
#include "kernels.cuh"
#include "philox.cuh"
#include "tcgen05.cuh"

namespace phi4 {

namespace tc {

constexpr int TILE = 128;            // particles per CTA = TMEM lanes
constexpr int STAGES = 4;            // Z ring depth; one stage = two K-steps (K = 16)
// ring stages per step filled by the epilogue warps (measured per C1 temperature: 0 -> 242 us,
// 1 -> 233, 2 -> 229, 3 -> 233)
constexpr int EPI_FILLS = 2;
static_assert(EPI_FILLS <= STAGES, "the epilogue fills of one step must fit the ring");
constexpr int EPI_PARTS = 4;         // warps per TMEM lane quarter (sites split four ways)
constexpr int EPI_WARPS = 4 * EPI_PARTS;
constexpr int PROD_WARPS = 8;
constexpr int PROD_WARP0 = EPI_WARPS;               // warps 16..23
constexpr int MMA_WARP = EPI_WARPS + PROD_WARPS;    // warp 24: the scheduler favours high warp ids
constexpr int THREADS = (EPI_WARPS + 1 + PROD_WARPS) * 32;   // 800
constexpr int CHUNK_BYTES = TILE * 16;           // one 16-byte K-chunk of all 128 rows
constexpr int SLAB_BYTES = 2 * 4 * CHUNK_BYTES;  // {hi,lo} x 4 K-chunks
constexpr int MAX_SMEM = 232448;

constexpr int ZSQ_BUFS = 4;          // IRMH: |z|^2 accumulators, one per step in flight
constexpr float ZSQ_SCALE = 4194304.f;   // 2^22: |z|^2 < 1024 in 32-bit fixed point, 2.4e-7 resolution
struct Smem {
  size_t tile0, tile1, lhi, llo, zring, part, dtab, bars, zsq, zzs, total;
};
__host__ __device__ inline Smem smem_layout(int V, bool irmh = false) {
  Smem s;
  size_t o = 0;
  const size_t tile = (size_t)V * TILE * 4, lmat = l_floats(V) * 4;
  s.tile0 = o; o += round_up((int)tile, 128);
  s.tile1 = o; o += round_up((int)tile, 128);
  s.lhi = o; o += round_up((int)lmat, 128);
  s.llo = o; o += round_up((int)lmat, 128);
  s.zring = o; o += (size_t)STAGES * SLAB_BYTES;
  s.part = o; o += (size_t)EPI_PARTS * TILE * 8 + TILE * 4;   // partial (dS, dU0) per part and particle; ln u
  s.dtab = o; o += round_up(32 * (kp_of(V) >> 3), 128);   // per-K-step operand descriptors (32 B each)
  s.bars = o; o += 128;
  // IRMH (reading A15): |z|^2 per particle and step in fixed point (integer atomics: the sum does
  // not depend on the order of the six threads that draw a particle's normals), and its float copy
  s.zsq = o; if (irmh) o += (size_t)ZSQ_BUFS * TILE * 4;
  s.zzs = o; if (irmh) o += (size_t)TILE * 4;
  s.total = o;
  return s;
}

}  // namespace tc

struct TcParams {
  float* phi; float* S; float* U0;
  const float* Lsplit;         // [2][Kp/4][Vn][4]: s*Lc split hi/lo, UMMA K-major interleave layout
  Ctrl* ctrl;
  uint8_t* acc_out; float* margin_out;
  int N, ld, L, V, Vn, Kp;
  float m0sq, lam, kappa;
  int mode;
  uint64_t seed;
  uint32_t tag_prop, tag_acc, t0;
  int k, respect_done;
  PhiloxKeys rk;               // round keys of `seed` (constant-bank operands of the Philox XORs)
  const float* mu; float* W2;  // IRMH: proposal mean [V]; |Lc^-1 (phi - mu)|^2 per particle [ld]
  StepRecord* finish_rec;      // not null: the last CTA closes the temperature (finish_step_device)
  int finish_max_rec;
  HostPoll* finish_poll;
};

// (s Lc) -> hi/lo TF32 split in the layout the MMA reads.  K-step ks is a block of two 16-byte
// K-chunks over the rows [xs(ks), Vn): element (x, y), ks = y / 8, sits at float offset
//   8 rows_before(ks) + ((y % 8) / 4) (Vn - xs) 4 + (x - xs) 4 + y % 4
// of its part (hi, then lo after l_floats(V) floats).  Zero beyond V (the strict upper triangle
// inside a block is zero in Lc itself).
__global__ void lsplit_kernel(const float* __restrict__ Lc, int V, int Vn, int Kp, float s,
                              float* __restrict__ out, size_t lpart, const Ctrl* ctrl,
                              int respect_done) {
  pdl_enter();
  if (respect_done && ctrl->done) return;
  const size_t idx = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (idx >= (size_t)Kp * Vn) return;
  const int y = (int)(idx / Vn), x = (int)(idx - (size_t)y * Vn);
  const int ks = y >> 3, xs = tc::xs_of(ks);
  if (x < xs) return;
  float v = (x < V && y < V && y <= x) ? s * Lc[(size_t)x * V + y] : 0.f;
  float hi = tc::tf32_rna(v);
  float lo = tc::tf32_rna(v - hi);
  const int rows = Vn - xs;
  size_t o = (size_t)tc::rows_before(ks, Vn) * 8 + (size_t)((y & 7) >> 2) * rows * 4 +
             (size_t)(x - xs) * 4 + (y & 3);
  out[o] = hi;
  out[lpart + o] = lo;
}

// Per-site difference of Eq. 1 between phi' (a2; forward neighbours b2, c2) and phi (a; b, c) in
// the lattice-Laplacian form: on the periodic lattice
//   S_E = sum_x [ (2 kappa + m0^2/2) phi_x^2 + lambda phi_x^4 - kappa phi_x (phi_{x+1} + phi_{x+2}) ],
// which is Eq. 1 with the squares expanded (each site appears in four bonds; kappa = 1 for Eq. 1,
// Eq. 5 of PAPER.md:313 is this form).  The bond sum dB is kept apart and scaled once at the end.  With
// q = a2^2 - a^2 formed as (a2-a)(a2+a), the potential part does not cancel; the bond part
// a2 (b2+c2) - a (b+c) carries an fp32 rounding of ~3e-7 per site, 3e-6 over the V <= 112 sites
// of this kernel -- far inside the 1e-4 decision band.  (The generic path, used up to V = 4096,
// keeps the fully difference-based form.)
__device__ __forceinline__ void tc_site_diff(float a, float b, float c, float a2, float b2,
                                             float c2, float c2m, float lam, float& dS, float& dB,
                                             float& dU) {
  const float q = (a2 - a) * (a2 + a);
  dS = fmaf(q, fmaf(lam, fmaf(a2, a2, a * a), c2m), dS);
  dB = fmaf(a, b + c, dB);
  dB = fmaf(-a2, b2 + c2, dB);
  dU = fmaf(0.5f, q, dU);
}

// Differences of Eq. 1 / U0 over the lattice rows r = g, g + EPI_PARTS, ... of one particle
// (column `pr` of the site-major tiles).  LT > 0: the lattice size is a compile-time constant, a
// row is fully unrolled -- all 4 LT shared-memory loads of a row (immediate offsets) are in
// flight before the arithmetic.  LT = 0: any L, one site at a time.
template <int LT>
__device__ __forceinline__ void tc_stencil(const float* cur, const float* oth, int g, int Lrt,
                                           float c2m, float lam, float kap, float& dS, float& dU) {
  using namespace tc;
  if constexpr (LT > 0) {
    float s0 = 0.f, u0 = 0.f, s1 = 0.f, u1 = 0.f, b0 = 0.f, b1 = 0.f;
    for (int r = g; r < LT; r += EPI_PARTS) {
      const int rn = (r + 1 == LT) ? 0 : r + 1;
      const float* c0 = cur + r * LT * TILE; const float* c1 = cur + rn * LT * TILE;
      const float* o0 = oth + r * LT * TILE; const float* o1 = oth + rn * LT * TILE;
      float a[LT], a2[LT], d[LT], d2[LT];
#pragma unroll
      for (int c = 0; c < LT; ++c) {
        a[c] = c0[c * TILE]; a2[c] = o0[c * TILE];
        d[c] = c1[c * TILE]; d2[c] = o1[c * TILE];
      }
#pragma unroll
      for (int c = 0; c < LT; ++c) {
        constexpr int dummy = 0; (void)dummy;
        const int cn = (c + 1 == LT) ? 0 : c + 1;
        if (c & 1) tc_site_diff(a[c], a[cn], d[c], a2[c], a2[cn], d2[c], c2m, lam, s1, b1, u1);
        else tc_site_diff(a[c], a[cn], d[c], a2[c], a2[cn], d2[c], c2m, lam, s0, b0, u0);
      }
    }
    dS = fmaf(kap, b0 + b1, s0 + s1);
    dU = u0 + u1;
  } else {
    const int L = Lrt;
    float dB = 0.f;
    for (int r = g; r < L; r += EPI_PARTS) {
      const int rn = (r + 1 == L) ? 0 : r + 1;
      const float* c0 = cur + r * L * TILE; const float* c1 = cur + rn * L * TILE;
      const float* o0 = oth + r * L * TILE; const float* o1 = oth + rn * L * TILE;
      float a = c0[0], a2 = o0[0];
      for (int c = 0; c < L; ++c) {
        const int cn = (c + 1 == L) ? 0 : c + 1;
        float b = c0[cn * TILE], b2 = o0[cn * TILE];
        float d = c1[c * TILE], d2 = o1[c * TILE];
        tc_site_diff(a, b, d, a2, b2, d2, c2m, lam, dS, dB, dU);
        a = b;
        a2 = b2;
      }
    }
    dS = fmaf(kap, dB, dS);
  }
}

__device__ __forceinline__ void named_bar_sync(int id, int nthreads) {
  asm volatile("bar.sync %0, %1;" ::"r"(id), "r"(nthreads) : "memory");
}

// Warp roles (800 threads, one CTA per SM):
//   warps 0..15   epilogue.  Warp w serves TMEM lane quarter Q = w % 4 (the hardware lets a warp
//                 read only lanes 32 (w % 4) .. +31) and site part g = w / 4: the four warps of a
//                 quarter split the 16-column TMEM blocks and the lattice rows of their 32
//                 particles and meet at named barrier 1 + Q.
//   warps 16..23  normal producers: thread (particle row, half) draws two Philox quads per ring
//                 stage, two stages (four independent chains) per pass.
//   warp 24       one thread issues every tcgen05.mma and the bulk copy of Lc; the operand
//                 descriptors of all K-steps are tabulated once in shared memory by its 32 lanes.
// IRMH (NEXT row f2, reading A15): the proposal is mu + Lc z (the factor is packed with s = 1), the
// margin gains log q(phi) - log q(phi') = 1/2 |z|^2 - 1/2 |w|^2, and an accepted particle's |w|^2
// becomes |z|^2.  |z|^2 is summed where the normals are drawn.
// NG > 0 (small populations: nested-sampling walkers, C0, the paper's N = 5000): a CTA owns NG
// groups of 32 particles (NG = 1 or 2) instead of 128.  They sit in TMEM lanes 0 .. 32 NG - 1 (the
// other rows of the A operand stay zero), so only the four warps of a group's lane quarter can
// read its accumulator rows, but the proposal then lies in shared memory and the group's 16 / NG
// epilogue warps share the stencil rows, the ring fills and the tile copies of its 32 particles
// (lane = particle in every warp), and the producer threads draw 1 or 2 quads per pass instead of
// four: a step is a latency chain, and the chain gets shorter; more SMs take part.
template <int LT, bool IRMH, int NG>
__global__ void __launch_bounds__(tc::THREADS, 1) mutate_tc_kernel(const TcParams p) {
  constexpr bool NARROW = NG > 0;
  // programmatic dependent launch: barrier setup and the TMEM allocation touch nothing the
  // predecessor writes, so they run before the wait
  pdl_trigger();
  using namespace tc;
  extern __shared__ __align__(1024) uint8_t smem[];
  const Smem lay = smem_layout(p.V, IRMH);
  uint32_t* zsq = reinterpret_cast<uint32_t*>(smem + lay.zsq);
  float* tile0 = reinterpret_cast<float*>(smem + lay.tile0);
  float* tile1 = reinterpret_cast<float*>(smem + lay.tile1);
  float2* part = reinterpret_cast<float2*>(smem + lay.part);
  uint64_t* bars = reinterpret_cast<uint64_t*>(smem + lay.bars);
  // barrier slots: zfull[S] zempty[S] dfull[2] dempty[2] lfull, then the TMEM base slot
  const uint32_t bar0 = smem_u32(bars);
  auto zfull = [&](int s) { return bar0 + 8u * s; };
  auto zempty = [&](int s) { return bar0 + 8u * (STAGES + s); };
  auto dfull = [&](int b) { return bar0 + 8u * (2 * STAGES + b); };
  auto dempty = [&](int b) { return bar0 + 8u * (2 * STAGES + 2 + b); };
  const uint32_t lfull = bar0 + 8u * (2 * STAGES + 4);
  uint32_t* tmem_slot = reinterpret_cast<uint32_t*>(bars + 2 * STAGES + 5);

  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const int V = p.V, Vn = p.Vn, Kp = p.Kp, nk8 = Kp >> 3, nit = (nk8 + 1) >> 1;
  // the first nitE ring fills of every step are produced by the epilogue warps (one quad per
  // thread, two steps ahead), the other nitP by the dedicated producers (two quads per thread)
  const int nitE = min(EPI_FILLS, nit - 1), nitP = nit - nitE;
  const int i0 = blockIdx.x * (NARROW ? 32 * NG : TILE);
  uint32_t ncols = 32;
  while ((int)ncols < 2 * Vn) ncols <<= 1;

  if (warp == MMA_WARP && lane == 0) {
    for (int s = 0; s < STAGES; ++s) { mbar_init(zfull(s), EPI_WARPS); mbar_init(zempty(s), 1); }
    for (int b = 0; b < 2; ++b) { mbar_init(dfull(b), 1); mbar_init(dempty(b), EPI_WARPS); }
    mbar_init(lfull, 1);
    fence_mbar_init();
  }
  if (warp == 0) tmem_alloc(smem_u32(tmem_slot), ncols);
  if (IRMH)
    for (int e = threadIdx.x; e < ZSQ_BUFS * TILE; e += THREADS) zsq[e] = 0u;
  if (NARROW) {            // rows 32 NG..127 of every ring stage are never written again: zero once
    float4* z4 = reinterpret_cast<float4*>(smem + lay.zring);
    for (int e = threadIdx.x; e < STAGES * SLAB_BYTES / 16; e += THREADS) z4[e] = make_float4(0.f, 0.f, 0.f, 0.f);
    fence_proxy_async();
  }
  tc_fence_before();
  __syncthreads();
  tc_fence_after();
  const uint32_t taddr = *tmem_slot;
  pdl_wait();
  if (p.respect_done && p.ctrl->done) {
    if (warp == 0) tmem_dealloc(taddr, ncols);
    return;
  }

  if (warp == MMA_WARP) {
    // ================================ MMA issuer (one thread) =================================
    // per-K-step table: {b_hi, b_lo, idesc, first row xs}; lane ks fills entry ks
    struct KStep { uint64_t b_hi, b_lo; uint32_t idesc, xs, pad0, pad1; };
    KStep* tab = reinterpret_cast<KStep*>(smem + lay.dtab);
    {
      const uint32_t lhi = smem_u32(smem + lay.lhi), llo = smem_u32(smem + lay.llo);
      for (int ks = lane; ks < nk8; ks += 32) {
        const int xs = xs_of(ks);
        const uint32_t lbo_b = (uint32_t)(Vn - xs) * 16;
        const uint32_t boff = (uint32_t)rows_before(ks, Vn) * 32;
        KStep e;
        e.b_hi = smem_desc(lhi + boff, lbo_b, 128);
        e.b_lo = smem_desc(llo + boff, lbo_b, 128);
        e.idesc = instr_desc(TILE, Vn - xs);
        e.xs = (uint32_t)xs; e.pad0 = 0; e.pad1 = 0;
        tab[ks] = e;
      }
    }
    __syncwarp();
    if (lane == 0) {
      const uint32_t lbytes = (uint32_t)l_floats(V) * 4;
      mbar_expect_tx(lfull, 2 * lbytes);
      bulk_g2s(smem_u32(smem + lay.lhi), p.Lsplit, lbytes, lfull);
      bulk_g2s(smem_u32(smem + lay.llo), p.Lsplit + l_floats(V), lbytes, lfull);
      mbar_wait(lfull, 0);
      // A descriptors differ only in the start address: slot s, K-step kk, hi / lo part
      const uint64_t a_base = smem_desc(smem_u32(smem + lay.zring), CHUNK_BYTES, 128);
      int s = 0;
      uint32_t ph = 0;
      for (int t = 0; t < p.k; ++t) {
        const int buf = t & 1;
        mbar_wait(dempty(buf), ((t >> 1) & 1) ^ 1);
        tc_fence_after();
        const uint32_t dbase = taddr + (uint32_t)(buf * Vn);
        for (int it = 0; it < nit; ++it) {
          const KStep e0 = tab[2 * it];
          const KStep e1 = tab[min(2 * it + 1, nk8 - 1)];
          const uint64_t a0 = a_base + (uint64_t)((uint32_t)s * (SLAB_BYTES >> 4));
          mbar_wait(zfull(s), ph);
          tc_fence_after();
          // the first K-step (xs = 0) overwrites all Vn columns; later ones accumulate
          tc_mma_tf32(dbase + e0.xs, a0 + (4 * CHUNK_BYTES >> 4), e0.b_hi, e0.idesc, it > 0);
          tc_mma_tf32(dbase + e0.xs, a0, e0.b_lo, e0.idesc, 1);
          tc_mma_tf32(dbase + e0.xs, a0, e0.b_hi, e0.idesc, 1);
          if (2 * it + 1 < nk8) {
            const uint64_t a1 = a0 + (2 * CHUNK_BYTES >> 4);
            tc_mma_tf32(dbase + e1.xs, a1 + (4 * CHUNK_BYTES >> 4), e1.b_hi, e1.idesc, 1);
            tc_mma_tf32(dbase + e1.xs, a1, e1.b_lo, e1.idesc, 1);
            tc_mma_tf32(dbase + e1.xs, a1, e1.b_hi, e1.idesc, 1);
          }
          tc_commit(zempty(s));
          if (++s == STAGES) { s = 0; ph ^= 1; }
        }
        tc_commit(dfull(buf));
      }
    }
    __syncwarp();
  } else if (warp >= PROD_WARP0) {
    // ================================ normal producers =======================================
    if constexpr (NARROW) {
      // thread (particle row, sub): 8 / TPR quads per pass (a pass = two ring stages of four
      // 16-byte K-chunks), TPR = threads per row; all quads of a thread lie in ONE stage, so a
      // stage is written by four warps.  EVERY producer warp waits for and arrives at EVERY
      // producer stage, writer or not: a parity wait only tells "one phase behind" from "level",
      // and a warp that skipped the stages of the other four could meet a slot two phases on
      // (its wait then passes at once, and it overwrites a stage the MMA has not read).
      constexpr int TP = 32 * (NG > 0 ? NG : 1), TPR = 256 / TP, QPT = 8 / TPR;
      const int j = threadIdx.x - PROD_WARP0 * 32;       // 0..255
      const int pr = j % TP, sub = j / TP, so = (sub * QPT) >> 2;
      const int i = i0 + pr;
      const int nq = (V + 3) >> 2;
      uint8_t* zr = smem + lay.zring;
      for (int t = 0; t < p.k; ++t) {
        const uint32_t tt = p.t0 + (uint32_t)t;
        for (int it = 0; it < nitP; it += 2) {
          const bool mine = it + so < nitP;               // (warp-uniform: so is)
          float4 hv[QPT], lv[QPT];
          if (mine) {
#pragma unroll
            for (int u = 0; u < QPT; ++u) {
              const int c = (sub * QPT + u) & 3, q = 4 * (nitE + it + so) + c;
              float z[4] = {0.f, 0.f, 0.f, 0.f};
              if (i < p.N && q < nq) {
                const U4 w = philox4x32_10_rk((uint32_t)q, (uint32_t)i, tt, p.tag_prop, p.rk);
                box_muller_fast(w.x, w.y, z[0], z[1]);
                box_muller_fast(w.z, w.w, z[2], z[3]);
              }
              hv[u].x = tf32_rna(z[0]); lv[u].x = z[0] - hv[u].x;  hv[u].y = tf32_rna(z[1]); lv[u].y = z[1] - hv[u].y;
              hv[u].z = tf32_rna(z[2]); lv[u].z = z[2] - hv[u].z;  hv[u].w = tf32_rna(z[3]); lv[u].w = z[3] - hv[u].w;
            }
          }
#pragma unroll
          for (int st2 = 0; st2 < 2; ++st2) {
            if (it + st2 >= nitP) break;
            const int n = t * nit + nitE + it + st2, sl = n % STAGES;
            const uint32_t ph = (uint32_t)(n / STAGES) & 1u;
            mbar_wait_relaxed(zempty(sl), ph ^ 1);
            if (st2 == so) {
#pragma unroll
              for (int u = 0; u < QPT; ++u) {
                const int c = (sub * QPT + u) & 3;
                uint8_t* st = zr + (size_t)sl * SLAB_BYTES + (size_t)c * CHUNK_BYTES + (size_t)pr * 16;
                *reinterpret_cast<float4*>(st) = hv[u];
                *reinterpret_cast<float4*>(st + 4 * CHUNK_BYTES) = lv[u];
              }
              fence_proxy_async();
            }
            __syncwarp();
            if (lane == 0) mbar_arrive_n(zfull(sl), 2);     // 8 warps x 2 = the 16 expected
          }
        }
      }
    } else {
      const int j = threadIdx.x - PROD_WARP0 * 32;         // 0..255
      const int pr = j & (TILE - 1), half = j >> 7;
      const int i = i0 + pr;
      const int nq = (V + 3) >> 2;
      uint8_t* zr = smem + lay.zring;
      for (int t = 0; t < p.k; ++t) {
        const uint32_t tt = p.t0 + (uint32_t)t;
        // two ring stages (four Philox chains) per pass: the chains are independent, so their
        // latencies overlap inside the warp
        for (int it = 0; it < nitP; it += 2) {
          const bool second = it + 1 < nitP;
          U4 w[4];
          bool ok[4];
  #pragma unroll
          for (int c = 0; c < 4; ++c) {
            const int q = 4 * (nitE + it + (c >> 1)) + 2 * (c & 1) + half;   // slab nitE + it + c/2, chunk 2 (c%2) + half
            ok[c] = (i < p.N) && (q < nq) && (c < 2 || second);
          }
          if (second) {
  #pragma unroll
            for (int c = 0; c < 4; ++c)
              w[c] = philox4x32_10_rk((uint32_t)(4 * (nitE + it + (c >> 1)) + 2 * (c & 1) + half), (uint32_t)i, tt, p.tag_prop, p.rk);
          } else {
  #pragma unroll
            for (int c = 0; c < 2; ++c)
              w[c] = philox4x32_10_rk((uint32_t)(4 * (nitE + it) + 2 * c + half), (uint32_t)i, tt, p.tag_prop, p.rk);
            w[2] = w[0]; w[3] = w[1];
          }
  #pragma unroll
          for (int st2 = 0; st2 < 2; ++st2) {
            if (st2 == 1 && !second) break;
            float4 hv[2], lv[2];
            float zz = 0.f;
  #pragma unroll
            for (int e = 0; e < 2; ++e) {
              const int c = 2 * st2 + e;
              float z[4] = {0.f, 0.f, 0.f, 0.f};
              if (ok[c]) {
                box_muller_fast(w[c].x, w[c].y, z[0], z[1]);
                box_muller_fast(w[c].z, w[c].w, z[2], z[3]);
              }
              if (IRMH) {                                  // R1: a ragged last quad is truncated at V
                const int x0 = 4 * (4 * (nitE + it + (c >> 1)) + 2 * (c & 1) + half);
  #pragma unroll
                for (int m = 0; m < 4; ++m) if (x0 + m < V) zz = fmaf(z[m], z[m], zz);
              }
              // hi = rna_tf32(z); lo = z - hi is exact and |lo| <= 2^-12 |z|: the tensor core's own
              // truncation of lo to 11 bits costs 2^-23 |z|, below the dropped lo*lo term
              hv[e].x = tf32_rna(z[0]); lv[e].x = z[0] - hv[e].x;
              hv[e].y = tf32_rna(z[1]); lv[e].y = z[1] - hv[e].y;
              hv[e].z = tf32_rna(z[2]); lv[e].z = z[2] - hv[e].z;
              hv[e].w = tf32_rna(z[3]); lv[e].w = z[3] - hv[e].w;
            }
            const int n = t * nit + nitE + it + st2, s = n % STAGES;    // ring slot and use of fill n
            const uint32_t ph = (uint32_t)(n / STAGES) & 1u;
            mbar_wait_relaxed(zempty(s), ph ^ 1);
            uint8_t* st = zr + (size_t)s * SLAB_BYTES + (size_t)half * CHUNK_BYTES + (size_t)pr * 16;
            *reinterpret_cast<float4*>(st) = hv[0];
            *reinterpret_cast<float4*>(st + 2 * CHUNK_BYTES) = hv[1];
            *reinterpret_cast<float4*>(st + 4 * CHUNK_BYTES) = lv[0];
            *reinterpret_cast<float4*>(st + 6 * CHUNK_BYTES) = lv[1];
            if (IRMH) atomicAdd(&zsq[(t & (ZSQ_BUFS - 1)) * TILE + pr], __float2uint_rn(zz * ZSQ_SCALE));
            fence_proxy_async();
            __syncwarp();
            if (lane == 0) mbar_arrive_n(zfull(s), 2);         // 8 warps x 2 = the 16 expected
          }
        }
      }
    }
  } else {
    // ================================ epilogue ==============================================
    if constexpr (NARROW) {
      // ---- group gq of 32 particles: lane = particle in each of its WPG warps; warp e16 of the group
      constexpr int NGc = NG > 0 ? NG : 1, WPG = EPI_WARPS / NGc;
      const int Q = warp & 3, g = warp >> 2, gq = Q % NGc, e16 = g * (4 / NGc) + Q / NGc;
      const int pr = 32 * gq + lane, i = i0 + pr;
      const bool live = i < p.N;
      const int L = LT > 0 ? LT : p.L;
      const float hm = 2.0f * p.kappa + 0.5f * p.m0sq, lam = p.lam, kap = p.kappa;
      float* cur = tile0 + pr;
      float* oth = tile1 + pr;
      for (int x = e16; x < V; x += WPG) cur[x * TILE] = live ? p.phi[(size_t)x * p.ld + i] : 0.f;
      float Si = live ? p.S[i] : 0.f, Ui = live ? p.U0[i] : 0.f;
      const float beta = (float)p.ctrl->beta, S_star = (float)p.ctrl->S_star;
      unsigned nacc = 0;
      const uint32_t tlane = taddr + ((uint32_t)(32 * gq) << 16);   // TMEM lanes of the group
      const int NB_ALL = 6 + gq;                            // named barrier of the group's warps
      named_bar_sync(NB_ALL, 32 * WPG);
      float* lus = reinterpret_cast<float*>(part + EPI_PARTS * TILE);
      uint8_t* zr = smem + lay.zring;
      const int nq = (V + 3) >> 2;
      // ring fills of step t by the epilogue warps: stage `it` (< nitE <= 2), chunk e16 & 3 by the
      // group's warps with e16 < 8 and e16 >> 2 == it; every warp arrives once per stage (the barrier
      // expects all sixteen)
      auto fill = [&](int t) {
        for (int it = 0; it < nitE; ++it) {
          const int n = t * nit + it, sl = n % STAGES;
          const uint32_t ph = (uint32_t)(n / STAGES) & 1u;
          mbar_wait_relaxed(zempty(sl), ph ^ 1);       // (every arriver: the slot's last use is over)
          if (e16 < 8 && (e16 >> 2) == it) {
            const int q = 4 * it + (e16 & 3);
            float z[4] = {0.f, 0.f, 0.f, 0.f};
            if (live && q < nq) {
              const U4 w = philox4x32_10_rk((uint32_t)q, (uint32_t)i, p.t0 + (uint32_t)t, p.tag_prop, p.rk);
              box_muller_fast(w.x, w.y, z[0], z[1]);
              box_muller_fast(w.z, w.w, z[2], z[3]);
            }
            float4 hv, lv;
            hv.x = tf32_rna(z[0]); lv.x = z[0] - hv.x;  hv.y = tf32_rna(z[1]); lv.y = z[1] - hv.y;
            hv.z = tf32_rna(z[2]); lv.z = z[2] - hv.z;  hv.w = tf32_rna(z[3]); lv.w = z[3] - hv.w;
            uint8_t* st = zr + (size_t)sl * SLAB_BYTES + (size_t)(e16 & 3) * CHUNK_BYTES + (size_t)pr * 16;
            *reinterpret_cast<float4*>(st) = hv;
            *reinterpret_cast<float4*>(st + 4 * CHUNK_BYTES) = lv;
            fence_proxy_async();
          }
          __syncwarp();
          if (lane == 0) mbar_arrive(zfull(sl));
        }
      };
      fill(0);
      if (p.k > 1) fill(1);
      for (int t = 0; t < p.k; ++t) {
        const int buf = t & 1;
        mbar_wait_relaxed(dfull(buf), (t >> 1) & 1);
        tc_fence_after();
        // pass 1 (the four warps of the group's lane quarter): phi' = phi + d on 16-column blocks
        if (Q == gq) {
          for (int cb = 16 * g; cb < Vn; cb += 32 * EPI_PARTS) {
            uint32_t r0[16], r1[16];
            const int cb1 = cb + 16 * EPI_PARTS;
            const bool two = cb1 < Vn;
            tmem_ld16(tlane + (uint32_t)(buf * Vn + cb), r0);
            if (two) tmem_ld16(tlane + (uint32_t)(buf * Vn + cb1), r1);
            tmem_ld_wait();
            const float* ci = cur + cb * TILE; float* oi = oth + cb * TILE;
#pragma unroll
            for (int jj = 0; jj < 16; ++jj)
              if (cb + jj < V) oi[jj * TILE] = ci[jj * TILE] + __uint_as_float(r0[jj]);
            if (two) {
              ci = cur + cb1 * TILE; oi = oth + cb1 * TILE;
#pragma unroll
              for (int jj = 0; jj < 16; ++jj)
                if (cb1 + jj < V) oi[jj * TILE] = ci[jj * TILE] + __uint_as_float(r1[jj]);
            }
          }
        }
        tc_fence_before();
        __syncwarp();
        if (lane == 0) mbar_arrive(dempty(buf));
        named_bar_sync(NB_ALL, 32 * WPG);              // the proposal of the 32 particles is in smem
        // pass 2: lattice rows e16, e16 + WPG, ... of every particle
        float dS = 0.f, dU = 0.f;
        {
          float dB = 0.f;
          for (int r = e16; r < L; r += WPG) {
            const int rn = (r + 1 == L) ? 0 : r + 1;
            const float* c0 = cur + r * L * TILE; const float* c1 = cur + rn * L * TILE;
            const float* o0 = oth + r * L * TILE; const float* o1 = oth + rn * L * TILE;
            if constexpr (LT > 0) {
              float a[LT], a2[LT], d[LT], d2[LT];
#pragma unroll
              for (int c = 0; c < LT; ++c) {
                a[c] = c0[c * TILE]; a2[c] = o0[c * TILE];
                d[c] = c1[c * TILE]; d2[c] = o1[c * TILE];
              }
#pragma unroll
              for (int c = 0; c < LT; ++c) {
                const int cn = (c + 1 == LT) ? 0 : c + 1;
                tc_site_diff(a[c], a[cn], d[c], a2[c], a2[cn], d2[c], hm, lam, dS, dB, dU);
              }
            } else {
              float a = c0[0], a2 = o0[0];
              for (int c = 0; c < L; ++c) {
                const int cn = (c + 1 == L) ? 0 : c + 1;
                const float b = c0[cn * TILE], b2 = o0[cn * TILE];
                tc_site_diff(a, b, c1[c * TILE], a2, b2, o1[c * TILE], hm, lam, dS, dB, dU);
                a = b;
                a2 = b2;
              }
            }
          }
          dS = fmaf(kap, dB, dS);
        }
        // WPG partials per particle: part[(gq WPG + e16) 32 + lane] (the 4 x 128 slots of the wide layout)
        part[(gq * WPG + e16) * 32 + lane] = make_float2(dS, dU);
        if (e16 == WPG - 1) lus[pr] = log_uniform(p.seed, p.tag_acc, p.t0 + (uint32_t)t, (uint32_t)i);
        named_bar_sync(NB_ALL, 32 * WPG);
        dS = 0.f; dU = 0.f;
#pragma unroll
        for (int m = 0; m < WPG; ++m) {
          const float2 v = part[(gq * WPG + m) * 32 + lane];
          dS += v.x;
          dU += v.y;
        }
        const float lu = lus[pr];
        float margin;
        bool acc;
        if (p.mode == MODE_SMC) {
          margin = -(dU + beta * dS) - lu;
          acc = margin > 0.f;
        } else {
          margin = -dU - lu;
          acc = (margin > 0.f) && (Si + dS < S_star);
        }
        acc = acc && live;
        if (acc) {
          float* tmp = cur; cur = oth; oth = tmp;
          Si += dS;
          Ui += dU;
          ++nacc;
        }
        if (live && e16 == 0) {
          if (p.acc_out) p.acc_out[(size_t)t * p.N + i] = (uint8_t)acc;
          if (p.margin_out) p.margin_out[(size_t)t * p.N + i] = margin;
        }
        if (t + 2 < p.k) fill(t + 2);
      }
      if (live) {
        for (int x = e16; x < V; x += WPG) p.phi[(size_t)x * p.ld + i] = cur[x * TILE];
        if (e16 == 0) { p.S[i] = Si; p.U0[i] = Ui; }
      }
      if (e16 == 0) {
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) nacc += __shfl_xor_sync(0xffffffffu, nacc, o);
        if (lane == 0 && nacc) atomicAdd(&p.ctrl->n_accept, nacc);
        if (lane == 0) __threadfence();
      }
    } else {
      const int Q = warp & 3, g = warp >> 2;       // lane quarter, site part
      const int pr = Q * 32 + lane;                // particle row = TMEM lane
      const int i = i0 + pr;
      const bool live = i < p.N;
      const int L = LT > 0 ? LT : p.L;
      const float hm = 2.0f * p.kappa + 0.5f * p.m0sq, lam = p.lam, kap = p.kappa;   // coefficient of phi^2 in the Laplacian form
      float* cur = tile0 + pr;
      float* oth = tile1 + pr;
      for (int x = g; x < V; x += EPI_PARTS) cur[x * TILE] = live ? p.phi[(size_t)x * p.ld + i] : 0.f;
      float Si = live ? p.S[i] : 0.f, Ui = live ? p.U0[i] : 0.f;
      float Wi = (IRMH && live) ? p.W2[i] : 0.f;          // |Lc^-1 (phi - mu)|^2 of the current state
      float* zzs = reinterpret_cast<float*>(smem + lay.zzs);
      const float beta = (float)p.ctrl->beta, S_star = (float)p.ctrl->S_star;
      unsigned nacc = 0;
      const uint32_t tlane = taddr + ((uint32_t)(Q * 32) << 16);
      named_bar_sync(1 + Q, 32 * EPI_PARTS);
      float* lus = reinterpret_cast<float*>(part + EPI_PARTS * TILE);
      uint8_t* zr = smem + lay.zring;
      const int nq = (V + 3) >> 2;
      // this thread's share of the normals of step t: quad 4 it + g of its own particle row
      auto fill = [&](int t) {
        // two stages per pass: both Philox chains first, then the maps and the stores
        for (int e0 = 0; e0 < nitE; e0 += 2) {
          U4 w[2];
  #pragma unroll
          for (int e = 0; e < 2; ++e)
            if (e0 + e < nitE) w[e] = philox4x32_10_rk((uint32_t)(4 * (e0 + e) + g), (uint32_t)i, p.t0 + (uint32_t)t, p.tag_prop, p.rk);
  #pragma unroll
          for (int e = 0; e < 2; ++e) {
            if (e0 + e >= nitE) break;
            const int it = e0 + e, q = 4 * it + g;
            float z[4] = {0.f, 0.f, 0.f, 0.f};
            if (live && q < nq) {
              box_muller_fast(w[e].x, w[e].y, z[0], z[1]);
              box_muller_fast(w[e].z, w[e].w, z[2], z[3]);
            }
            if (IRMH) {                                    // R1: a ragged last quad is truncated at V
              float zz = 0.f;
  #pragma unroll
              for (int m = 0; m < 4; ++m) if (4 * q + m < V) zz = fmaf(z[m], z[m], zz);
              atomicAdd(&zsq[(t & (ZSQ_BUFS - 1)) * TILE + pr], __float2uint_rn(zz * ZSQ_SCALE));
            }
            float4 hv, lv;
            hv.x = tf32_rna(z[0]); lv.x = z[0] - hv.x;  hv.y = tf32_rna(z[1]); lv.y = z[1] - hv.y;
            hv.z = tf32_rna(z[2]); lv.z = z[2] - hv.z;  hv.w = tf32_rna(z[3]); lv.w = z[3] - hv.w;
            const int n = t * nit + it, s = n % STAGES;
            const uint32_t ph = (uint32_t)(n / STAGES) & 1u;
            mbar_wait_relaxed(zempty(s), ph ^ 1);
            uint8_t* st = zr + (size_t)s * SLAB_BYTES + (size_t)g * CHUNK_BYTES + (size_t)pr * 16;
            *reinterpret_cast<float4*>(st) = hv;
            *reinterpret_cast<float4*>(st + 4 * CHUNK_BYTES) = lv;
            fence_proxy_async();
            __syncwarp();
            if (lane == 0) mbar_arrive(zfull(s));
          }
        }
      };
      // the epilogue warps produce the FIRST slabs of a step and run two steps ahead: the MMAs of
      // step t + 1 then never wait for a warp that is itself waiting for the MMAs of step t
      fill(0);
      if (p.k > 1) fill(1);
      for (int t = 0; t < p.k; ++t) {
        const int buf = t & 1;
        mbar_wait_relaxed(dfull(buf), (t >> 1) & 1);
        tc_fence_after();
        // pass 1: phi' = phi + d on this part's 16-column blocks (d carries the step scale s); two
        // TMEM loads in flight per wait
        for (int cb = 16 * g; cb < Vn; cb += 32 * EPI_PARTS) {
          uint32_t r0[16], r1[16];
          const int cb1 = cb + 16 * EPI_PARTS;
          const bool two = cb1 < Vn;
          tmem_ld16(tlane + (uint32_t)(buf * Vn + cb), r0);
          if (two) tmem_ld16(tlane + (uint32_t)(buf * Vn + cb1), r1);
          tmem_ld_wait();
          const float* ci = cur + cb * TILE; float* oi = oth + cb * TILE;
          if (cb + 16 <= V) {
  #pragma unroll
            for (int jj = 0; jj < 16; ++jj) oi[jj * TILE] = (IRMH ? __ldg(p.mu + cb + jj) : ci[jj * TILE]) + __uint_as_float(r0[jj]);
          } else {
  #pragma unroll
            for (int jj = 0; jj < 16; ++jj)
              if (cb + jj < V) oi[jj * TILE] = (IRMH ? __ldg(p.mu + cb + jj) : ci[jj * TILE]) + __uint_as_float(r0[jj]);
          }
          if (two) {
            ci = cur + cb1 * TILE; oi = oth + cb1 * TILE;
            if (cb1 + 16 <= V) {
  #pragma unroll
              for (int jj = 0; jj < 16; ++jj) oi[jj * TILE] = (IRMH ? __ldg(p.mu + cb1 + jj) : ci[jj * TILE]) + __uint_as_float(r1[jj]);
            } else {
  #pragma unroll
              for (int jj = 0; jj < 16; ++jj)
                if (cb1 + jj < V) oi[jj * TILE] = (IRMH ? __ldg(p.mu + cb1 + jj) : ci[jj * TILE]) + __uint_as_float(r1[jj]);
            }
          }
        }
        tc_fence_before();
        __syncwarp();
        if (lane == 0) mbar_arrive(dempty(buf));
        named_bar_sync(1 + Q, 32 * EPI_PARTS);       // the whole proposal of these 32 particles is in smem
        // pass 2: per-site differences of Eq. 1 and U0 over this part's lattice rows
        float dS = 0.f, dU = 0.f;
        tc_stencil<LT>(cur, oth, g, L, hm, lam, kap, dS, dU);
        part[g * TILE + pr] = make_float2(dS, dU);
        if (g == EPI_PARTS - 1) {
          lus[pr] = log_uniform(p.seed, p.tag_acc, p.t0 + (uint32_t)t, (uint32_t)i);
          if (IRMH) {                                  // |z|^2 of this step; the slot is free again
            uint32_t* zq = &zsq[(t & (ZSQ_BUFS - 1)) * TILE + pr];
            zzs[pr] = (float)*zq * (1.0f / ZSQ_SCALE);
            *zq = 0u;
          }
        }
        named_bar_sync(1 + Q, 32 * EPI_PARTS);
        // every part sums the four partials in the same order and takes the same decision (M4)
        dS = 0.f; dU = 0.f;
  #pragma unroll
        for (int m = 0; m < EPI_PARTS; ++m) {
          float2 v = part[m * TILE + pr];
          dS += v.x;
          dU += v.y;
        }
        const float lu = lus[pr];
        float margin;
        bool acc;
        float tZ = 0.f;
        if (IRMH) {
          tZ = zzs[pr];
          margin = -(dU + beta * dS) + 0.5f * (tZ - Wi) - lu;
          acc = margin > 0.f;
        } else if (p.mode == MODE_SMC) {
          margin = -(dU + beta * dS) - lu;
          acc = margin > 0.f;
        } else {
          margin = -dU - lu;
          acc = (margin > 0.f) && (Si + dS < S_star);
        }
        acc = acc && live;
        if (acc) {
          float* tmp = cur; cur = oth; oth = tmp;
          Si += dS;
          Ui += dU;
          if (IRMH) Wi = tZ;
          ++nacc;
        }
        if (live && g == 0) {
          if (p.acc_out) p.acc_out[(size_t)t * p.N + i] = (uint8_t)acc;
          if (p.margin_out) p.margin_out[(size_t)t * p.N + i] = margin;
        }
        if (t + 2 < p.k) fill(t + 2);
      }
      if (live) {
        for (int x = g; x < V; x += EPI_PARTS) p.phi[(size_t)x * p.ld + i] = cur[x * TILE];
        if (g == 0) { p.S[i] = Si; p.U0[i] = Ui; if (IRMH) p.W2[i] = Wi; }
      }
      if (g == 0) {
  #pragma unroll
        for (int o = 16; o > 0; o >>= 1) nacc += __shfl_xor_sync(0xffffffffu, nacc, o);
        if (lane == 0 && nacc) atomicAdd(&p.ctrl->n_accept, nacc);
        if (lane == 0) __threadfence();
      }
  
    }
  }
  tc_fence_before();
  __syncthreads();
  if (warp == 0) tmem_dealloc(taddr, ncols);
  if (p.finish_rec && threadIdx.x == 0) {
    // the CTA that counts in last has seen every other CTA's acceptances (fence, then counter)
    __threadfence();
    if (atomicAdd(&p.ctrl->cta_done, 1u) == gridDim.x - 1) {
      __threadfence();
      p.ctrl->cta_done = 0u;
      finish_step_device(p.ctrl, p.finish_rec, p.finish_max_rec, p.k, p.N, p.finish_poll);
    }
  }
}

bool mutate_tc_supported(int V, bool irmh) {
  return V >= 1 && tc::vn_of(V) <= 256 && tc::smem_layout(V, irmh).total <= (size_t)tc::MAX_SMEM;
}

size_t mutate_tc_lsplit_floats(int V) { return 2 * tc::l_floats(V); }

// Packed hi / lo split of s*Lc with Vn rows (>= V, multiple of 16) and Kp columns (>= V, multiple
// of 8); the lo part starts l_floats_vk(Vn, Kp) floats after the hi part.
void launch_lsplit(const float* Lc, int V, int Vn, int Kp, float s, float* Lsplit, const Ctrl* ctrl,
                   int respect_done, cudaStream_t st) {
  ++g_launches;
  launch_pdl(lsplit_kernel, (unsigned)(((size_t)Kp * Vn + 255) / 256), 256, 0, st, 
      Lc, V, Vn, Kp, s, Lsplit, tc::l_floats_vk(Vn, Kp), ctrl, respect_done);
}

void launch_mutate_tc(const MutateArgs& a, float* Lsplit, cudaStream_t st, const float* mu, float* W2) {
  const int V = a.md.V, Vn = tc::vn_of(V), Kp = tc::kp_of(V);
  const bool irmh = mu != nullptr;                 // independent proposal mu + Lc z: no step scale
  launch_lsplit(a.Lc, V, Vn, Kp, irmh ? 1.0f : a.s, Lsplit, a.ctrl, a.respect_done, st);
  TcParams p;
  p.phi = a.phi; p.S = a.S; p.U0 = a.U0; p.Lsplit = Lsplit; p.ctrl = a.ctrl;
  p.acc_out = a.acc_out; p.margin_out = a.margin_out;
  p.N = a.N; p.ld = a.ld; p.L = a.md.L; p.V = V; p.Vn = Vn; p.Kp = Kp;
  p.m0sq = a.md.m0sq; p.lam = a.md.lam; p.kappa = a.md.kappa; p.mode = a.mode; p.seed = a.seed;
  p.tag_prop = a.tag_prop; p.tag_acc = a.tag_acc; p.t0 = a.t0; p.k = a.k;
  p.respect_done = a.respect_done;
  p.mu = mu; p.W2 = W2;
  p.finish_rec = a.finish_rec; p.finish_max_rec = a.finish_max_rec; p.finish_poll = a.finish_poll;
  p.rk = philox_round_keys(a.seed);
  const size_t smem = tc::smem_layout(V, irmh).total;
  // at most one wave of 32- or 64-particle CTAs: the narrow variants (nested-sampling walkers, C0,
  // the paper's N = 5000)
  const int ng = irmh ? 0 : (a.ld / 32 <= 148 ? 1 : (a.ld / 64 <= 148 ? 2 : 0));
  static bool attr_done = false;
  if (!attr_done) {
    auto big = [](auto kern) { cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, tc::MAX_SMEM); };
    big(mutate_tc_kernel<0, false, 0>); big(mutate_tc_kernel<4, false, 0>); big(mutate_tc_kernel<10, false, 0>);
    big(mutate_tc_kernel<0, true, 0>); big(mutate_tc_kernel<10, true, 0>);
    big(mutate_tc_kernel<0, false, 1>); big(mutate_tc_kernel<4, false, 1>); big(mutate_tc_kernel<10, false, 1>);
    big(mutate_tc_kernel<0, false, 2>); big(mutate_tc_kernel<4, false, 2>); big(mutate_tc_kernel<10, false, 2>);
    attr_done = true;
  }
  const dim3 grid(ng ? a.ld / (32 * ng) : a.ld / tc::TILE);
  ++g_launches;
  // lattice sizes of the BASELINE configs get a fully unrolled stencil; any other L the loop
  auto go = [&](auto k0, auto k4, auto k10) {
    if (p.L == 10) launch_pdl(k10, grid, tc::THREADS, smem, st, p);
    else if (p.L == 4) launch_pdl(k4, grid, tc::THREADS, smem, st, p);
    else launch_pdl(k0, grid, tc::THREADS, smem, st, p);
  };
  if (irmh) go(mutate_tc_kernel<0, true, 0>, mutate_tc_kernel<0, true, 0>, mutate_tc_kernel<10, true, 0>);
  else if (ng == 1) go(mutate_tc_kernel<0, false, 1>, mutate_tc_kernel<4, false, 1>, mutate_tc_kernel<10, false, 1>);
  else if (ng == 2) go(mutate_tc_kernel<0, false, 2>, mutate_tc_kernel<4, false, 2>, mutate_tc_kernel<10, false, 2>);
  else go(mutate_tc_kernel<0, false, 0>, mutate_tc_kernel<4, false, 0>, mutate_tc_kernel<10, false, 0>);
}

}  // namespace phi4
