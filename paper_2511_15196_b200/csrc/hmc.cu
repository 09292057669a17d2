// hmc.cu -- NEXT row f1: HMC rejuvenation inside SMC (PAPER.md:53(iii), :172: "short HMC
// trajectories", "diagonal mass matrix", "fixed trajectory of 20 leapfrog steps"; reading A14).
//
// Target U(phi) = U0 + beta S_E.  Mass matrix M = diag(1/var_x), var_x = the particle variance of
// site x (diagonal of the covariance of reading A4); momentum p = z / sqrt(var), z = PROP-stream
// normals.  One transition: half kick, nfrog x (drift phi += eps var p, kick p -= eps grad U, the
// last kick halved), then g = (H_old - H_new) - ln u, accept iff g > 0.
//
// No dense contraction here (the diagonal mass matrix makes the drift elementwise): the kernel is
// bound by the FP32 pipe.  A CTA owns 32 particles for all k transitions; lane = particle, warp w
// owns a band of lattice rows (two by default) whose position, momentum and eps*var live in REGISTERS for the
// whole trajectory (the lattice side is a template parameter, every index is a compile-time
// constant).  East/west neighbours come from registers, the two halo rows from a double-buffered
// site-major [V][32] shared-memory tile into which every band publishes its rows after each
// drift: one barrier, ~1 LDS + 1 STS and ~11 FP32 instructions per site per leapfrog step.
// HBM traffic: phi read and written once per temperature.
#include "kernels.cuh"
#include "philox.cuh"

namespace phi4 {

namespace hm {
constexpr int P = 32;                       // particles per CTA (one per lane)
constexpr int MAX_L = 22;                   // three [V][32] fp32 tiles must fit in 200 KB
// Band height per lattice side (measured at L = 10 and 16: even bands of few, tall warps win --
// fewer halo rows and barrier partners -- as long as a thread's 3 x R x LT values stay in
// registers): the tallest even split with R * LT <= 64 sites per thread, else the least ragged.
__host__ __device__ constexpr int rows_per_band(int LT) {
  constexpr int tab[23] = {1, 1, 2, 3, 4, 5, 6, 7, 8, 3, 5, 4, 4, 2, 2, 3, 4, 2, 3, 3, 3, 3, 2};
  return tab[LT];
}
__host__ __device__ constexpr int bands(int LT) {
  return (LT + rows_per_band(LT) - 1) / rows_per_band(LT);
}
}  // namespace hm

struct HmcArgs {
  float* phi; float* S; float* U0; const float* Sigma;
  int N, ld; Model md; float eps; int nfrog;
  uint64_t seed; uint32_t t0; int k; Ctrl* ctrl;
  uint8_t* acc_out; float* margin_out; int respect_done;
};

// bands of different height run different instantiations of the same barrier sequence
__device__ __forceinline__ void cta_sync() { asm volatile("bar.sync 0;" ::: "memory"); }

// p -= h * grad U on a band of NR rows.  hn / hs: this lane's column of the halo rows north of
// the band's first row and south of its last row (stride P per site).
template <int LT, int NR, int R>
__device__ __forceinline__ void hmc_kick(const float (&q)[R * LT], float (&p)[R * LT],
                                         const float* hn, const float* hs, float h, float beta,
                                         float m0sq, float lam4, float kap) {
#pragma unroll
  for (int jr = 0; jr < NR; ++jr)
#pragma unroll
    for (int c = 0; c < LT; ++c) {
      const int j = jr * LT + c;
      const float a = q[j];
      const float e = q[jr * LT + (c + 1) % LT], w = q[jr * LT + (c + LT - 1) % LT];
      const float n = jr == 0 ? hn[c * hm::P] : q[jr == 0 ? j : j - LT];
      const float s = jr == NR - 1 ? hs[c * hm::P] : q[jr == NR - 1 ? j : j + LT];
      // grad S_E = (4 a - neighbours) + m0^2 a + 4 lambda a^3;  grad U = a + beta grad S_E
      const float gs = fmaf(kap, fmaf(4.0f, a, -((e + w) + (n + s))), a * fmaf(lam4, a * a, m0sq));
      p[j] = fmaf(-h, fmaf(beta, gs, a), p[j]);
    }
}

template <int LT, int NR>
__device__ __forceinline__ void hmc_band(const HmcArgs& A, float* cur, float* hal0, float* hal1,
                                         const float* var_s, const float* isd_s, float4* red,
                                         int* flag) {
  using namespace hm;
  constexpr int V = LT * LT, NB = bands(LT), R = rows_per_band(LT), NS = NR * LT;
  constexpr int nq = (V + 3) >> 2;
  const int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
  const int i = blockIdx.x * P + lane;
  const bool live = i < A.N;
  const int r0 = w * R, x0 = r0 * LT;
  const int rn = (r0 + LT - 1) % LT, rs = (r0 + NR) % LT;       // halo rows
  const float beta = (float)A.ctrl->beta, m0sq = A.md.m0sq, lam = A.md.lam, lam4 = 4.0f * A.md.lam,
              kap = A.md.kappa, hk = 0.5f * A.md.kappa;
  const float eps = A.eps;
  float q[R * LT], p[R * LT], ev[R * LT];
#pragma unroll
  for (int j = 0; j < NS; ++j) ev[j] = eps * var_s[x0 + j];
  float Si = live ? A.S[i] : 0.f, Ui = live ? A.U0[i] : 0.f;
  unsigned nacc = 0;
  float* const own0 = hal0 + x0 * P + lane;
  float* const own1 = hal1 + x0 * P + lane;
  float* const ownc = cur + x0 * P + lane;
#pragma unroll
  for (int j = 0; j < NS; ++j) q[j] = live ? A.phi[(size_t)(x0 + j) * A.ld + i] : 0.f;
#pragma unroll
  for (int j = 0; j < NS; ++j) ownc[j * P] = q[j];

  for (int jt = 0; jt < A.k; ++jt) {
    const uint32_t t = A.t0 + (uint32_t)jt;
    // momentum normals by quad (shared evenly between the bands), staged in hal1
    for (int qd = w; qd < nq; qd += NB) {
      float z[4] = {0.f, 0.f, 0.f, 0.f};
      if (live) normals4(A.seed, TAG_PROP, t, (uint32_t)i, (uint32_t)qd, z);
#pragma unroll
      for (int e = 0; e < 4; ++e)
        if (4 * qd + e < V) hal1[(4 * qd + e) * P + lane] = z[e];
    }
#pragma unroll
    for (int j = 0; j < NS; ++j) {
      q[j] = ownc[j * P];
      own0[j * P] = q[j];
    }
    cta_sync();
    float K0 = 0.f;
#pragma unroll
    for (int j = 0; j < NS; ++j) {
      const float z = own1[j * P];
      p[j] = z * isd_s[x0 + j];
      K0 = fmaf(0.5f * z, z, K0);
    }
    hmc_kick<LT, NR, R>(q, p, hal0 + rn * LT * P + lane, hal0 + rs * LT * P + lane, 0.5f * eps, beta,
                     m0sq, lam4, kap);
    cta_sync();                       // hal1 (the staged normals) is free from here on
    for (int s = 0; s < A.nfrog; ++s) {
      float* const own = (s & 1) ? own0 : own1;
      const float* const hb = (s & 1) ? hal0 : hal1;
#pragma unroll
      for (int j = 0; j < NS; ++j) {
        q[j] = fmaf(ev[j], p[j], q[j]);
        own[j * P] = q[j];
      }
      cta_sync();
      hmc_kick<LT, NR, R>(q, p, hb + rn * LT * P + lane, hb + rs * LT * P + lane,
                       (s + 1 == A.nfrog) ? 0.5f * eps : eps, beta, m0sq, lam4, kap);
    }
    // H_new: kinetic, S_E (Eq. 1, forward neighbours), U0 over this band
    const float* const hs = (((A.nfrog - 1) & 1) ? hal0 : hal1) + rs * LT * P + lane;
    float K1 = 0.f, Sp = 0.f, Up = 0.f;
#pragma unroll
    for (int jr = 0; jr < NR; ++jr) {
      float rowS = 0.f;
#pragma unroll
      for (int c = 0; c < LT; ++c) {
        const int j = jr * LT + c;
        const float a = q[j], b = q[jr * LT + (c + 1) % LT];
        const float d = jr == NR - 1 ? hs[c * P] : q[jr == NR - 1 ? j : j + LT];
        const float e1 = b - a, e2 = d - a, a2 = a * a;
        rowS += hk * (e1 * e1 + e2 * e2) + a2 * (0.5f * m0sq + lam * a2);
        Up = fmaf(0.5f, a2, Up);
        K1 = fmaf(0.5f * ev[j] * p[j], p[j], K1);
      }
      Sp += rowS;
    }
    red[w * P + lane] = make_float4(K0, K1 / eps, Sp, Up);       // ev = eps * var
    cta_sync();
    if (w == 0) {
      float4 tot = make_float4(0.f, 0.f, 0.f, 0.f);
#pragma unroll
      for (int m = 0; m < NB; ++m) {
        const float4 v = red[m * P + lane];
        tot.x += v.x; tot.y += v.y; tot.z += v.z; tot.w += v.w;
      }
      int acc = 0;
      if (live) {
        const float lu = log_uniform(A.seed, TAG_ACC, t, (uint32_t)i);
        // (H_old - H_new) - ln u with the differences taken term by term
        const float margin = ((Ui - tot.w) + beta * (Si - tot.z) + (tot.x - tot.y)) - lu;
        acc = margin > 0.f;
        if (acc) { Si = tot.z; Ui = tot.w; ++nacc; }
        if (A.acc_out) A.acc_out[(size_t)jt * A.N + i] = (uint8_t)acc;
        if (A.margin_out) A.margin_out[(size_t)jt * A.N + i] = margin;
      }
      flag[lane] = acc;
    }
    cta_sync();
    if (flag[lane]) {
#pragma unroll
      for (int j = 0; j < NS; ++j) ownc[j * P] = q[j];
    }
    // the next transition's staging writes hal1 / own0, which every warp finished reading before
    // the barrier above; flag[] is rewritten only two barriers further on
  }
  if (live) {
#pragma unroll
    for (int j = 0; j < NS; ++j) A.phi[(size_t)(x0 + j) * A.ld + i] = ownc[j * P];
    if (w == 0) { A.S[i] = Si; A.U0[i] = Ui; }
  }
  if (w == 0) {
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) nacc += __shfl_xor_sync(0xffffffffu, nacc, o);
    if (lane == 0 && nacc) atomicAdd(&A.ctrl->n_accept, nacc);
  }
}

template <int LT>
__global__ void __launch_bounds__(32 * hm::bands(LT)) hmc_kernel(const HmcArgs A) {
  using namespace hm;
  constexpr int V = LT * LT, NB = bands(LT), R = rows_per_band(LT);
  extern __shared__ __align__(16) float sm[];
  __shared__ int flag[P];
  if (A.respect_done && A.ctrl->done) return;
  float4* red = reinterpret_cast<float4*>(sm);   // [NB][32] partial (K0, K1, S', U0')
  float* cur = sm + 4 * NB * P;                  // [V][32] current particles
  float* hal0 = cur + V * P;                     // [V][32] published positions, double-buffered
  float* hal1 = hal0 + V * P;
  float* var_s = hal1 + V * P;                   // [V]
  float* isd_s = var_s + V;                      // [V] 1/sqrt(var)
  const int w = threadIdx.x >> 5;
  for (int x = threadIdx.x; x < V; x += 32 * NB) {
    const float v = A.Sigma[(size_t)x * V + x];
    var_s[x] = v;
    isd_s[x] = rsqrtf(v);
  }
  cta_sync();
  constexpr int LAST = LT - (NB - 1) * R;        // height of the last band
  if (LAST != R && w == NB - 1)
    hmc_band<LT, LAST>(A, cur, hal0, hal1, var_s, isd_s, red, flag);
  else
    hmc_band<LT, R>(A, cur, hal0, hal1, var_s, isd_s, red, flag);
}

static size_t hmc_smem_bytes(int L) {
  const int V = L * L;
  return ((size_t)3 * V * hm::P + 2 * V) * sizeof(float) +
         (size_t)hm::bands(L) * hm::P * sizeof(float4);
}

bool hmc_supported(int V) {
  int L = 1;
  while (L * L < V) ++L;
  return L * L == V && L <= hm::MAX_L;
}

template <int LT>
static void launch_hmc_lt(const HmcArgs& a, cudaStream_t st) {
  static bool attr_done = false;
  if (!attr_done) {
    cudaFuncSetAttribute(hmc_kernel<LT>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                         (int)hmc_smem_bytes(LT));
    attr_done = true;
  }
  hmc_kernel<LT><<<(a.N + hm::P - 1) / hm::P, 32 * hm::bands(LT), hmc_smem_bytes(LT), st>>>(a);
}

template <int LT>
static void dispatch_hmc(const HmcArgs& a, cudaStream_t st) {
  if (a.md.L == LT) launch_hmc_lt<LT>(a, st);
  else if constexpr (LT > 1) dispatch_hmc<LT - 1>(a, st);
}

void launch_hmc(float* phi, float* S, float* U0, const float* Sigma, int N, int ld, Model md,
                float eps, int nfrog, uint64_t seed, uint32_t t0, int k, Ctrl* ctrl,
                uint8_t* acc_out, float* margin_out, int respect_done, cudaStream_t st) {
  HmcArgs a{phi, S, U0, Sigma, N, ld, md, eps, nfrog, seed, t0, k, ctrl, acc_out, margin_out,
            respect_done};
  ++g_launches;
  dispatch_hmc<hm::MAX_L>(a, st);
}

}  // namespace phi4

// ---------------------------------------------------------------------------------------------
// Any lattice size: the fields of a trajectory no longer fit on one SM (L > 22), so position and
// momentum live in HBM scratch ([V][ld] each, positions double-buffered) and every leapfrog step
// is its own launch (the stencil needs the neighbours' updated positions: a grid-wide
// dependency): a kick and the drift after it in one pass.  HBM-bound: 16 B per site per leapfrog
// step.  Same arithmetic, streams and reading A14 as hmc_kernel.
namespace phi4 {

// momentum refresh, q <- phi, K0 = 1/2 sum z^2.  Block = 32 particles x 8 quad groups.
__global__ void __launch_bounds__(256)
hmc_g_init_kernel(const float* __restrict__ phi, float* __restrict__ q, float* __restrict__ p,
                  const float* __restrict__ Sigma, float* __restrict__ K0, int N, int ld, int V,
                  uint64_t seed, uint32_t t, const Ctrl* ctrl, int respect_done) {
  if (respect_done && ctrl->done) return;
  __shared__ float part[8][32];
  const int lane = threadIdx.x & 31, g = threadIdx.x >> 5;
  const int i = blockIdx.x * 32 + lane;
  const int nq = (V + 3) >> 2;
  float k0 = 0.f;
  if (i < N) {
    for (int qd = g; qd < nq; qd += 8) {
      float z[4];
      normals4(seed, TAG_PROP, t, (uint32_t)i, (uint32_t)qd, z);
#pragma unroll
      for (int e = 0; e < 4; ++e) {
        const int x = 4 * qd + e;
        if (x < V) {
          const size_t o = (size_t)x * ld + i;
          p[o] = z[e] * rsqrtf(Sigma[(size_t)x * V + x]);
          q[o] = phi[o];
          k0 = fmaf(0.5f * z[e], z[e], k0);
        }
      }
    }
  }
  part[g][lane] = k0;
  __syncthreads();
  if (g == 0 && i < N) {
    float a = 0.f;
#pragma unroll
    for (int m = 0; m < 8; ++m) a += part[m][lane];
    K0[i] = a;
  }
}

// p -= h grad U(q): one thread per (site, particle); blockIdx.y = site
__global__ void __launch_bounds__(256)
hmc_g_kick_kernel(const float* __restrict__ q, float* __restrict__ p, int N, int ld, Model md,
                  float h, const Ctrl* ctrl, int respect_done) {
  if (respect_done && ctrl->done) return;
  const int i = blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= N) return;
  const int L = md.L, x = blockIdx.y, r = x / L, c = x - r * L;
  const int ce = c + 1 == L ? 0 : c + 1, cw = c == 0 ? L - 1 : c - 1;
  const int rs = r + 1 == L ? 0 : r + 1, rn = r == 0 ? L - 1 : r - 1;
  const float a = q[(size_t)x * ld + i];
  const float e = q[(size_t)(r * L + ce) * ld + i], w = q[(size_t)(r * L + cw) * ld + i];
  const float n = q[(size_t)(rn * L + c) * ld + i], s = q[(size_t)(rs * L + c) * ld + i];
  const float beta = (float)ctrl->beta;
  const float gs = fmaf(md.kappa, fmaf(4.0f, a, -((e + w) + (n + s))), a * fmaf(4.0f * md.lam, a * a, md.m0sq));
  const size_t o = (size_t)x * ld + i;
  p[o] = fmaf(-h, fmaf(beta, gs, a), p[o]);
}

// Kick and the drift that follows it in one pass: p -= h grad U(q_in); q_out = q_in + eps var p.
// The drift must not overwrite positions that other threads still read as neighbours, so q is
// double-buffered; the arithmetic is that of the two separate kernels, bit for bit.  16 B per
// site and leapfrog step instead of 24 (the path is HBM-bound).
__global__ void __launch_bounds__(256)
hmc_g_kickdrift_kernel(const float* __restrict__ qin, float* __restrict__ qout, float* __restrict__ p,
                       const float* __restrict__ Sigma, int N, int ld, Model md, float h, float eps,
                       const Ctrl* ctrl, int respect_done) {
  if (respect_done && ctrl->done) return;
  const int i = blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= N) return;
  const int L = md.L, V = md.V, x = blockIdx.y, r = x / L, c = x - r * L;
  const int ce = c + 1 == L ? 0 : c + 1, cw = c == 0 ? L - 1 : c - 1;
  const int rs = r + 1 == L ? 0 : r + 1, rn = r == 0 ? L - 1 : r - 1;
  const float a = qin[(size_t)x * ld + i];
  const float e = qin[(size_t)(r * L + ce) * ld + i], w = qin[(size_t)(r * L + cw) * ld + i];
  const float n = qin[(size_t)(rn * L + c) * ld + i], s = qin[(size_t)(rs * L + c) * ld + i];
  const float beta = (float)ctrl->beta;
  const float gs = fmaf(md.kappa, fmaf(4.0f, a, -((e + w) + (n + s))), a * fmaf(4.0f * md.lam, a * a, md.m0sq));
  const size_t o = (size_t)x * ld + i;
  const float pn = fmaf(-h, fmaf(beta, gs, a), p[o]);
  p[o] = pn;
  qout[o] = fmaf(eps * Sigma[(size_t)x * V + x], pn, a);
}

// H_new, margin, accept, commit.  Block = 32 particles x 8 row groups (as accept_kernel).
__global__ void __launch_bounds__(256)
hmc_g_accept_kernel(float* __restrict__ phi, const float* __restrict__ q,
                    const float* __restrict__ p, const float* __restrict__ Sigma,
                    const float* __restrict__ K0, float* __restrict__ S, float* __restrict__ U0,
                    int N, int ld, Model md, uint64_t seed, uint32_t t, Ctrl* ctrl,
                    uint8_t* __restrict__ acc_out, float* __restrict__ margin_out,
                    int respect_done) {
  if (respect_done && ctrl->done) return;
  __shared__ float ps[8][32], pu[8][32], pk[8][32];
  __shared__ int flag[32];
  const int lane = threadIdx.x & 31, g = threadIdx.x >> 5;
  const int i = blockIdx.x * 32 + lane;
  const int L = md.L, V = md.V;
  const float hm = 0.5f * md.m0sq, lam = md.lam, hk = 0.5f * md.kappa;
  const int band = (L + 7) >> 3, r_lo = min(L, g * band), r_hi = min(L, r_lo + band);
  float Sp = 0.f, Up = 0.f, K1 = 0.f;
  if (i < N) {
    for (int r = r_lo; r < r_hi; ++r) {
      const int rs = r + 1 == L ? 0 : r + 1;
      float rowS = 0.f, rowU = 0.f, rowK = 0.f;       // two-level fp32 accumulation
      float a = q[(size_t)(r * L) * ld + i];
      for (int c = 0; c < L; ++c) {
        const int x = r * L + c, ce = c + 1 == L ? 0 : c + 1;
        const float b = q[(size_t)(r * L + ce) * ld + i], d = q[(size_t)(rs * L + c) * ld + i];
        const float pp = p[(size_t)x * ld + i];
        const float e1 = b - a, e2 = d - a, a2 = a * a;
        rowS += hk * (e1 * e1 + e2 * e2) + a2 * (hm + lam * a2);
        rowU = fmaf(0.5f, a2, rowU);
        rowK = fmaf(0.5f * Sigma[(size_t)x * V + x] * pp, pp, rowK);
        a = b;
      }
      Sp += rowS; Up += rowU; K1 += rowK;
    }
  }
  ps[g][lane] = Sp; pu[g][lane] = Up; pk[g][lane] = K1;
  __syncthreads();
  if (g == 0) {
    int acc = 0;
    if (i < N) {
      float tS = 0.f, tU = 0.f, tK = 0.f;
#pragma unroll
      for (int m = 0; m < 8; ++m) { tS += ps[m][lane]; tU += pu[m][lane]; tK += pk[m][lane]; }
      const float lu = log_uniform(seed, TAG_ACC, t, (uint32_t)i);
      const float Si = S[i], Ui = U0[i];
      const float margin = ((Ui - tU) + (float)ctrl->beta * (Si - tS) + (K0[i] - tK)) - lu;
      acc = margin > 0.f;
      if (acc) { S[i] = tS; U0[i] = tU; }
      if (acc_out) acc_out[i] = (uint8_t)acc;
      if (margin_out) margin_out[i] = margin;
    }
    flag[lane] = acc;
    const unsigned m = __ballot_sync(0xffffffffu, acc);
    if (lane == 0 && m) atomicAdd(&ctrl->n_accept, (unsigned)__popc(m));
  }
  __syncthreads();
  if (i < N && flag[lane]) {
    for (int r = r_lo; r < r_hi; ++r)
      for (int c = 0; c < L; ++c) {
        const size_t o = (size_t)(r * L + c) * ld + i;
        phi[o] = q[o];
      }
  }
}

// q, q2, p: [V][ld] scratch each; K0: [ld] scratch
void launch_hmc_generic(float* phi, float* S, float* U0, const float* Sigma, float* q, float* q2,
                        float* p, float* K0, int N, int ld, Model md, float eps, int nfrog, uint64_t seed,
                        uint32_t t0, int k, Ctrl* ctrl, uint8_t* acc_out, float* margin_out,
                        int respect_done, cudaStream_t st) {
  const int V = md.V;
  const dim3 gs((N + 255) / 256, V);
  for (int j = 0; j < k; ++j) {
    const uint32_t t = t0 + (uint32_t)j;
    ++g_launches;
    hmc_g_init_kernel<<<ld / 32, 256, 0, st>>>(phi, q, p, Sigma, K0, N, ld, V, seed, t, ctrl, respect_done);
    // p -= eps/2 grad U; nfrog x { q += eps var p; p -= eps grad U (eps/2 after the last drift) }
    // as nfrog fused (kick, drift) passes between the two position buffers and one last kick
    float* qa = q;
    float* qb = q2;
    for (int s = 0; s < nfrog; ++s) {
      ++g_launches;
      hmc_g_kickdrift_kernel<<<gs, 256, 0, st>>>(qa, qb, p, Sigma, N, ld, md, s == 0 ? 0.5f * eps : eps, eps,
                                                 ctrl, respect_done);
      float* tmp = qa; qa = qb; qb = tmp;
    }
    ++g_launches;
    hmc_g_kick_kernel<<<gs, 256, 0, st>>>(qa, p, N, ld, md, 0.5f * eps, ctrl, respect_done);
    ++g_launches;
    hmc_g_accept_kernel<<<ld / 32, 256, 0, st>>>(
        phi, qa, p, Sigma, K0, S, U0, N, ld, md, seed, t, ctrl,
        acc_out ? acc_out + (size_t)j * N : nullptr, margin_out ? margin_out + (size_t)j * N : nullptr,
        respect_done);
  }
}

}  // namespace phi4
