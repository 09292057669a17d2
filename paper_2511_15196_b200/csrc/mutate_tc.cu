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

namespace phi4 {

namespace tc {

constexpr int TILE = 128;            // particles per CTA = TMEM lanes
constexpr int STAGES = 4;            // Z ring depth (K-steps in flight)
constexpr int EPI_WARPS = 4;
constexpr int PROD_WARPS = 8;
constexpr int MMA_WARP = EPI_WARPS;  // warp 4
constexpr int THREADS = (EPI_WARPS + 1 + PROD_WARPS) * 32;
constexpr int SLAB_BYTES = 2 * 2 * TILE * 16;   // {hi,lo} x 2 K-chunks x 128 rows x 16 B
constexpr int MAX_SMEM = 232448;

__host__ __device__ inline int vn_of(int V) { return round_up(V, 16); }
__host__ __device__ inline int kp_of(int V) { return round_up(V, 8); }

struct Smem {
  size_t tile0, tile1, lhi, llo, zring, bars, total;
};
__host__ __device__ inline Smem smem_layout(int V) {
  Smem s;
  size_t o = 0;
  const size_t tile = (size_t)V * TILE * 4, lmat = (size_t)kp_of(V) * vn_of(V) * 4;
  s.tile0 = o; o += round_up((int)tile, 128);
  s.tile1 = o; o += round_up((int)tile, 128);
  s.lhi = o; o += round_up((int)lmat, 128);
  s.llo = o; o += round_up((int)lmat, 128);
  s.zring = o; o += (size_t)STAGES * SLAB_BYTES;
  s.bars = o; o += 256;
  s.total = o;
  return s;
}

// ------------------------------------------------------------------ PTX wrappers -------------
__device__ __forceinline__ uint32_t smem_u32(const void* p) {
  return (uint32_t)__cvta_generic_to_shared(p);
}
__device__ __forceinline__ void mbar_init(uint32_t bar, uint32_t count) {
  asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(bar), "r"(count));
}
__device__ __forceinline__ void mbar_arrive(uint32_t bar) {
  asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(bar) : "memory");
}
__device__ __forceinline__ void mbar_expect_tx(uint32_t bar, uint32_t bytes) {
  asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(bar), "r"(bytes)
               : "memory");
}
__device__ __forceinline__ void mbar_wait(uint32_t bar, uint32_t parity) {
  asm volatile(
      "{\n\t"
      ".reg .pred p;\n\t"
      "WAIT_%=:\n\t"
      "mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n\t"
      "@p bra DONE_%=;\n\t"
      "bra WAIT_%=;\n\t"
      "DONE_%=:\n\t"
      "}" ::"r"(bar), "r"(parity)
      : "memory");
}
__device__ __forceinline__ void fence_proxy_async() {
  asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
}
__device__ __forceinline__ void fence_mbar_init() {
  asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
}
__device__ __forceinline__ void bulk_g2s(uint32_t dst, const void* src, uint32_t bytes,
                                         uint32_t bar) {
  asm volatile(
      "cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];" ::
          "r"(dst), "l"(src), "r"(bytes), "r"(bar)
      : "memory");
}
__device__ __forceinline__ void tc_fence_before() {
  asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory");
}
__device__ __forceinline__ void tc_fence_after() {
  asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
}
__device__ __forceinline__ void tmem_alloc(uint32_t slot, uint32_t ncols) {
  asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], %1;" ::"r"(slot),
               "r"(ncols)
               : "memory");
  asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;" ::: "memory");
}
__device__ __forceinline__ void tmem_dealloc(uint32_t taddr, uint32_t ncols) {
  asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, %1;" ::"r"(taddr), "r"(ncols)
               : "memory");
}
__device__ __forceinline__ void tc_commit(uint32_t bar) {
  asm volatile("tcgen05.commit.cta_group::1.mbarrier::arrive::one.shared::cluster.b64 [%0];" ::
                   "r"(bar)
               : "memory");
}
// D[tmem] (+)= A[smem] * B[smem]^T, kind::tf32, one CTA.
__device__ __forceinline__ void tc_mma_tf32(uint32_t d, uint64_t a, uint64_t b, uint32_t idesc,
                                            uint32_t accumulate) {
  asm volatile(
      "{\n\t"
      ".reg .pred p;\n\t"
      "setp.ne.b32 p, %4, 0;\n\t"
      "tcgen05.mma.cta_group::1.kind::tf32 [%0], %1, %2, %3, p;\n\t"
      "}" ::"r"(d), "l"(a), "l"(b), "r"(idesc), "r"(accumulate)
      : "memory");
}
__device__ __forceinline__ void tmem_ld16(uint32_t taddr, uint32_t (&r)[16]) {
  asm volatile(
      "tcgen05.ld.sync.aligned.32x32b.x16.b32 "
      "{%0, %1, %2, %3, %4, %5, %6, %7, %8, %9, %10, %11, %12, %13, %14, %15}, [%16];"
      : "=r"(r[0]), "=r"(r[1]), "=r"(r[2]), "=r"(r[3]), "=r"(r[4]), "=r"(r[5]), "=r"(r[6]),
        "=r"(r[7]), "=r"(r[8]), "=r"(r[9]), "=r"(r[10]), "=r"(r[11]), "=r"(r[12]), "=r"(r[13]),
        "=r"(r[14]), "=r"(r[15])
      : "r"(taddr)
      : "memory");
  asm volatile("tcgen05.wait::ld.sync.aligned;" ::: "memory");
}

// Shared-memory matrix descriptor, K-major, no swizzle ("interleave"): core matrix = 8 rows x
// 16 B stored contiguously; LBO = byte distance between the two 16-byte K-chunks of one MMA,
// SBO = byte distance between 8-row groups.  (Field layout: start>>4 [0,14), LBO>>4 [16,30),
// SBO>>4 [32,46), version=1 [46,48), layout type 0 [61,64).)
__device__ __forceinline__ uint64_t smem_desc(uint32_t addr, uint32_t lbo, uint32_t sbo) {
  return (uint64_t)((addr >> 4) & 0x3FFFu) | ((uint64_t)((lbo >> 4) & 0x3FFFu) << 16) |
         ((uint64_t)((sbo >> 4) & 0x3FFFu) << 32) | (1ull << 46);
}
// Instruction descriptor: D = F32 [4,6)=1, A = B = TF32 [7,10)=[10,13)=2, both K-major,
// N>>3 at [17,23), M>>4 at [24,29).
__device__ __forceinline__ uint32_t instr_desc(int M, int N) {
  return (1u << 4) | (2u << 7) | (2u << 10) | ((uint32_t)(N >> 3) << 17) |
         ((uint32_t)(M >> 4) << 24);
}
__device__ __forceinline__ float tf32_rna(float x) {
  uint32_t u;
  asm("cvt.rna.tf32.f32 %0, %1;" : "=r"(u) : "f"(x));
  return __uint_as_float(u);
}

}  // namespace tc

struct TcParams {
  float* phi; float* S; float* U0;
  const float* Lsplit;         // [2][Kp/4][Vn][4]: s*Lc split hi/lo, UMMA K-major interleave layout
  Ctrl* ctrl;
  uint8_t* acc_out; float* margin_out;
  int N, ld, L, V, Vn, Kp;
  float m0sq, lam;
  int mode;
  uint64_t seed;
  uint32_t tag_prop, tag_acc, t0;
  int k, respect_done;
};

// (s Lc) -> hi/lo TF32 split in the layout the MMA reads: element (x, y) of part h at
// ((h*(Kp/4) + y/4) * Vn + x) * 4 + y%4; zero outside the lower triangle / beyond V.
__global__ void lsplit_kernel(const float* __restrict__ Lc, int V, int Vn, int Kp, float s,
                              float* __restrict__ out, const Ctrl* ctrl, int respect_done) {
  if (respect_done && ctrl->done) return;
  int idx = blockIdx.x * blockDim.x + threadIdx.x;
  if (idx >= Kp * Vn) return;
  int y = idx / Vn, x = idx - y * Vn;
  float v = (x < V && y < V && y <= x) ? s * Lc[(size_t)x * V + y] : 0.f;
  float hi = tc::tf32_rna(v);
  float lo = tc::tf32_rna(v - hi);
  size_t o = ((size_t)(y >> 2) * Vn + x) * 4 + (y & 3);
  out[o] = hi;
  out[(size_t)Kp * Vn + o] = lo;
}

__device__ __forceinline__ void tc_site_diff(float a, float b, float c, float a2, float b2,
                                             float c2, float hm, float lam, float& dS, float& dU) {
  float q = (a2 - a) * (a2 + a);
  float e = b - a, e2 = b2 - a2, f = c - a, f2 = c2 - a2;
  dS += 0.5f * ((e2 - e) * (e2 + e) + (f2 - f) * (f2 + f)) + q * (hm + lam * (a2 * a2 + a * a));
  dU += 0.5f * q;
}

__global__ void __launch_bounds__(tc::THREADS, 1) mutate_tc_kernel(const TcParams p) {
  using namespace tc;
  extern __shared__ __align__(1024) uint8_t smem[];
  if (p.respect_done && p.ctrl->done) return;
  const Smem lay = smem_layout(p.V);
  float* tile0 = reinterpret_cast<float*>(smem + lay.tile0);
  float* tile1 = reinterpret_cast<float*>(smem + lay.tile1);
  uint64_t* bars = reinterpret_cast<uint64_t*>(smem + lay.bars);
  // barrier slots: zfull[4] zempty[4] dfull[2] dempty[2] lfull, then the TMEM base slot
  const uint32_t bar0 = smem_u32(bars);
  auto zfull = [&](int s) { return bar0 + 8u * s; };
  auto zempty = [&](int s) { return bar0 + 8u * (STAGES + s); };
  auto dfull = [&](int b) { return bar0 + 8u * (2 * STAGES + b); };
  auto dempty = [&](int b) { return bar0 + 8u * (2 * STAGES + 2 + b); };
  const uint32_t lfull = bar0 + 8u * (2 * STAGES + 4);
  uint32_t* tmem_slot = reinterpret_cast<uint32_t*>(bars + 2 * STAGES + 5);

  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const int V = p.V, Vn = p.Vn, Kp = p.Kp, nk8 = Kp >> 3;
  const int i0 = blockIdx.x * TILE;
  uint32_t ncols = 32;
  while ((int)ncols < 2 * Vn) ncols <<= 1;

  if (warp == MMA_WARP && lane == 0) {
    for (int s = 0; s < STAGES; ++s) { mbar_init(zfull(s), PROD_WARPS); mbar_init(zempty(s), 1); }
    for (int b = 0; b < 2; ++b) { mbar_init(dfull(b), 1); mbar_init(dempty(b), EPI_WARPS); }
    mbar_init(lfull, 1);
    fence_mbar_init();
  }
  if (warp == 0) tmem_alloc(smem_u32(tmem_slot), ncols);
  tc_fence_before();
  __syncthreads();
  tc_fence_after();
  const uint32_t taddr = *tmem_slot;

  if (warp == MMA_WARP) {
    // ================================ MMA issuer (one thread) =================================
    if (lane == 0) {
      const uint32_t lbytes = (uint32_t)Kp * Vn * 4;
      mbar_expect_tx(lfull, 2 * lbytes);
      bulk_g2s(smem_u32(smem + lay.lhi), p.Lsplit, lbytes, lfull);
      bulk_g2s(smem_u32(smem + lay.llo), p.Lsplit + (size_t)Kp * Vn, lbytes, lfull);
      mbar_wait(lfull, 0);
      const uint32_t lhi = smem_u32(smem + lay.lhi), llo = smem_u32(smem + lay.llo);
      const uint32_t zr = smem_u32(smem + lay.zring);
      const uint32_t lbo_b = (uint32_t)Vn * 16;
      int s = 0;
      uint32_t ph = 0;
      for (int t = 0; t < p.k; ++t) {
        const int buf = t & 1;
        mbar_wait(dempty(buf), ((t >> 1) & 1) ^ 1);
        tc_fence_after();
        for (int ks = 0; ks < nk8; ++ks) {
          mbar_wait(zfull(s), ph);
          tc_fence_after();
          // rows x < 8 ks of this K-step are zero: start at the 16-aligned row below
          const int xs = (8 * ks) & ~15;
          const int n = Vn - xs;
          const uint32_t idesc = instr_desc(TILE, n);
          const uint32_t d = taddr + (uint32_t)(buf * Vn + xs);
          const uint32_t za = zr + (uint32_t)s * SLAB_BYTES;
          const uint64_t a_hi = smem_desc(za, TILE * 16, 128);
          const uint64_t a_lo = smem_desc(za + 2 * TILE * 16, TILE * 16, 128);
          const uint32_t boff = (uint32_t)(2 * ks) * lbo_b + (uint32_t)xs * 16;
          const uint64_t b_hi = smem_desc(lhi + boff, lbo_b, 128);
          const uint64_t b_lo = smem_desc(llo + boff, lbo_b, 128);
          // the first K-step (xs = 0) overwrites all Vn columns; later ones accumulate
          tc_mma_tf32(d, a_lo, b_hi, idesc, ks > 0);
          tc_mma_tf32(d, a_hi, b_lo, idesc, 1);
          tc_mma_tf32(d, a_hi, b_hi, idesc, 1);
          tc_commit(zempty(s));
          if (++s == STAGES) { s = 0; ph ^= 1; }
        }
        tc_commit(dfull(buf));
      }
    }
    __syncwarp();
  } else if (warp > MMA_WARP) {
    // ================================ normal producers =======================================
    const int j = threadIdx.x - (MMA_WARP + 1) * 32;     // 0..255
    const int pr = j & (TILE - 1), half = j >> 7;
    const int i = i0 + pr;
    const int nq = (V + 3) >> 2;
    uint8_t* zr = smem + lay.zring;
    int s = 0;
    uint32_t ph = 0;
    for (int t = 0; t < p.k; ++t) {
      for (int ks = 0; ks < nk8; ++ks) {
        const int q = 2 * ks + half;
        float z[4] = {0.f, 0.f, 0.f, 0.f};
        if (q < nq && i < p.N) normals4(p.seed, p.tag_prop, p.t0 + (uint32_t)t, (uint32_t)i, (uint32_t)q, z);
        float4 hi, lo;
        hi.x = tf32_rna(z[0]); lo.x = tf32_rna(z[0] - hi.x);
        hi.y = tf32_rna(z[1]); lo.y = tf32_rna(z[1] - hi.y);
        hi.z = tf32_rna(z[2]); lo.z = tf32_rna(z[2] - hi.z);
        hi.w = tf32_rna(z[3]); lo.w = tf32_rna(z[3] - hi.w);
        mbar_wait(zempty(s), ph ^ 1);
        uint8_t* slab = zr + (size_t)s * SLAB_BYTES + (size_t)half * (TILE * 16) + (size_t)pr * 16;
        *reinterpret_cast<float4*>(slab) = hi;
        *reinterpret_cast<float4*>(slab + 2 * TILE * 16) = lo;
        fence_proxy_async();
        __syncwarp();
        if (lane == 0) mbar_arrive(zfull(s));
        if (++s == STAGES) { s = 0; ph ^= 1; }
      }
    }
  } else {
    // ================================ epilogue: thread = particle =============================
    const int pr = threadIdx.x;                 // 0..127 = TMEM lane
    const int i = i0 + pr;
    const bool live = i < p.N;
    const int L = p.L;
    const float hm = 0.5f * p.m0sq, lam = p.lam;
    float* cur = tile0 + pr;
    float* oth = tile1 + pr;
    for (int x = 0; x < V; ++x) cur[x * TILE] = live ? p.phi[(size_t)x * p.ld + i] : 0.f;
    float Si = live ? p.S[i] : 0.f, Ui = live ? p.U0[i] : 0.f;
    const float beta = (float)p.ctrl->beta, S_star = (float)p.ctrl->S_star;
    unsigned nacc = 0;
    const uint32_t tlane = taddr + ((uint32_t)(warp * 32) << 16);
    for (int t = 0; t < p.k; ++t) {
      const int buf = t & 1;
      mbar_wait(dfull(buf), (t >> 1) & 1);
      tc_fence_after();
      // pass 1: phi' = phi + d  (d already carries the step scale s)
      for (int cb = 0; cb < Vn; cb += 16) {
        uint32_t r[16];
        tmem_ld16(tlane + (uint32_t)(buf * Vn + cb), r);
#pragma unroll
        for (int jj = 0; jj < 16; ++jj) {
          int x = cb + jj;
          if (x < V) oth[x * TILE] = cur[x * TILE] + __uint_as_float(r[jj]);
        }
      }
      tc_fence_before();
      __syncwarp();
      if (lane == 0) mbar_arrive(dempty(buf));
      // pass 2: per-site differences of Eq. 1 and U0
      float dS = 0.f, dU = 0.f;
      for (int r = 0; r < L; ++r) {
        const int rn = (r + 1 == L) ? 0 : r + 1;
        const float* c0 = cur + r * L * TILE; const float* c1 = cur + rn * L * TILE;
        const float* o0 = oth + r * L * TILE; const float* o1 = oth + rn * L * TILE;
        float a = c0[0], a2 = o0[0];
        for (int c = 0; c < L; ++c) {
          const int cn = (c + 1 == L) ? 0 : c + 1;
          float b = c0[cn * TILE], b2 = o0[cn * TILE];
          float d = c1[c * TILE], d2 = o1[c * TILE];
          tc_site_diff(a, b, d, a2, b2, d2, hm, lam, dS, dU);
          a = b;
          a2 = b2;
        }
      }
      // M4
      const float lu = log_uniform(p.seed, p.tag_acc, p.t0 + (uint32_t)t, (uint32_t)i);
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
      if (live) {
        if (p.acc_out) p.acc_out[(size_t)t * p.N + i] = (uint8_t)acc;
        if (p.margin_out) p.margin_out[(size_t)t * p.N + i] = margin;
      }
    }
    if (live) {
      for (int x = 0; x < V; ++x) p.phi[(size_t)x * p.ld + i] = cur[x * TILE];
      p.S[i] = Si;
      p.U0[i] = Ui;
    }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) nacc += __shfl_xor_sync(0xffffffffu, nacc, o);
    if (lane == 0 && nacc) atomicAdd(&p.ctrl->n_accept, nacc);
  }
  tc_fence_before();
  __syncthreads();
  if (warp == 0) tmem_dealloc(taddr, ncols);
}

bool mutate_tc_supported(int V) {
  return V >= 1 && tc::vn_of(V) <= 256 && tc::smem_layout(V).total <= (size_t)tc::MAX_SMEM;
}

size_t mutate_tc_lsplit_floats(int V) { return (size_t)2 * tc::kp_of(V) * tc::vn_of(V); }

void launch_mutate_tc(const MutateArgs& a, float* Lsplit, cudaStream_t st) {
  const int V = a.md.V, Vn = tc::vn_of(V), Kp = tc::kp_of(V);
  ++g_launches; lsplit_kernel<<<(Kp * Vn + 255) / 256, 256, 0, st>>>(a.Lc, V, Vn, Kp, a.s, Lsplit, a.ctrl,
                                                      a.respect_done);
  TcParams p;
  p.phi = a.phi; p.S = a.S; p.U0 = a.U0; p.Lsplit = Lsplit; p.ctrl = a.ctrl;
  p.acc_out = a.acc_out; p.margin_out = a.margin_out;
  p.N = a.N; p.ld = a.ld; p.L = a.md.L; p.V = V; p.Vn = Vn; p.Kp = Kp;
  p.m0sq = a.md.m0sq; p.lam = a.md.lam; p.mode = a.mode; p.seed = a.seed;
  p.tag_prop = a.tag_prop; p.tag_acc = a.tag_acc; p.t0 = a.t0; p.k = a.k;
  p.respect_done = a.respect_done;
  const size_t smem = tc::smem_layout(V).total;
  static bool attr_done = false;
  if (!attr_done) {
    cudaFuncSetAttribute(mutate_tc_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize,
                         tc::MAX_SMEM);
    attr_done = true;
  }
  ++g_launches; mutate_tc_kernel<<<a.ld / tc::TILE, tc::THREADS, smem, st>>>(p);
}

}  // namespace phi4
