// hmc.cu -- NEXT row f1: HMC rejuvenation inside SMC (PAPER.md:53(iii), :172: "short HMC
// trajectories", "diagonal mass matrix", "fixed trajectory of 20 leapfrog steps"; reading A14).
//
// Target U(phi) = U0 + beta S_E.  Mass matrix M = diag(1/var_x), var_x = the particle variance of
// site x (diagonal of the covariance of reading A4); momentum p = z / sqrt(var), z = PROP-stream
// normals.  One transition: half kick, nfrog x (drift phi += eps var p, kick p -= eps grad U, the
// last kick halved), then g = (H_old - H_new) - ln u, accept iff g > 0.
//
// No dense contraction here: the kernel is stencil / ALU bound.  A block owns 32 particles for all
// k transitions; phi, the trajectory position q and the momentum p live in shared memory as
// site-major [V][32] tiles (a warp reads 32 consecutive particles of one site: conflict free),
// eight warps split the lattice rows, two barriers per leapfrog step.  HBM traffic: phi read and
// written once per temperature.
#include "kernels.cuh"
#include "philox.cuh"

namespace phi4 {

namespace hm {
constexpr int P = 32, G = 8, THREADS = P * G;
}

__device__ __forceinline__ float hmc_grad_u(const float* q, int x, int r, int c, int L, float beta,
                                            float m0sq, float lam4) {
  const int cw = c == 0 ? L - 1 : c - 1, ce = c + 1 == L ? 0 : c + 1;
  const int rn = r == 0 ? L - 1 : r - 1, rs = r + 1 == L ? 0 : r + 1;
  const float a = q[x * hm::P];
  const float nb = q[(r * L + ce) * hm::P] + q[(r * L + cw) * hm::P] + q[(rs * L + c) * hm::P] +
                   q[(rn * L + c) * hm::P];
  // grad S_E = (4 a - neighbours) + m0^2 a + 4 lambda a^3;  grad U = a + beta grad S_E
  const float gs = fmaf(4.0f, a, -nb) + a * fmaf(lam4, a * a, m0sq);
  return fmaf(beta, gs, a);
}

__global__ void __launch_bounds__(hm::THREADS)
hmc_kernel(float* __restrict__ phi, float* __restrict__ S, float* __restrict__ U0,
           const float* __restrict__ Sigma, int N, int ld, Model md, float eps, int nfrog,
           uint64_t seed, uint32_t t0, int k, Ctrl* ctrl, uint8_t* __restrict__ acc_out,
           float* __restrict__ margin_out, int respect_done) {
  using namespace hm;
  extern __shared__ __align__(16) float sm[];
  if (respect_done && ctrl->done) return;
  const int V = md.V, L = md.L;
  float4* red = reinterpret_cast<float4*>(sm);   // [G][32] partial (K0, K1, S', U0')
  float* cur = sm + 4 * G * P;     // [V][32] current particles
  float* q = cur + V * P;          // trajectory position
  float* p = q + V * P;            // momentum
  float* var = p + V * P;          // [V]
  float* isd = var + V;            // [V] 1/sqrt(var)
  __shared__ int flag[P];
  const int lane = threadIdx.x & 31, g = threadIdx.x >> 5;
  const int i = blockIdx.x * P + lane;
  const bool live = i < N;
  const float beta = (float)ctrl->beta, m0sq = md.m0sq, lam = md.lam, lam4 = 4.0f * md.lam;
  const int nq = (V + 3) >> 2;

  for (int x = threadIdx.x; x < V; x += THREADS) {
    const float v = Sigma[(size_t)x * V + x];
    var[x] = v;
    isd[x] = rsqrtf(v);
  }
  for (int x = g; x < V; x += G) cur[x * P + lane] = live ? phi[(size_t)x * ld + i] : 0.f;
  float Si = live ? S[i] : 0.f, Ui = live ? U0[i] : 0.f;
  unsigned nacc = 0;
  __syncthreads();
  const float* cq = q + lane;
  for (int j = 0; j < k; ++j) {
    const uint32_t t = t0 + (uint32_t)j;
    // momentum refresh (quads q ~ g) and q <- cur (rows ~ g)
    float K0 = 0.f;
    for (int qd = g; qd < nq; qd += G) {
      float z[4] = {0.f, 0.f, 0.f, 0.f};
      if (live) normals4(seed, TAG_PROP, t, (uint32_t)i, (uint32_t)qd, z);
#pragma unroll
      for (int e = 0; e < 4; ++e) {
        const int x = 4 * qd + e;
        if (x < V) {
          p[x * P + lane] = z[e] * isd[x];
          K0 = fmaf(0.5f * z[e], z[e], K0);
        }
      }
    }
    for (int x = g; x < V; x += G) q[x * P + lane] = cur[x * P + lane];
    __syncthreads();
    // half kick
    for (int r = g; r < L; r += G)
      for (int c = 0; c < L; ++c) {
        const int x = r * L + c;
        p[x * P + lane] -= 0.5f * eps * hmc_grad_u(cq, x, r, c, L, beta, m0sq, lam4);
      }
    for (int s = 0; s < nfrog; ++s) {
      // other warps may still be reading this warp's rows of q in their kick
      __syncthreads();
      // drift on this warp's rows (only its own p), then everyone needs the new q
      for (int r = g; r < L; r += G)
        for (int c = 0; c < L; ++c) {
          const int x = r * L + c;
          q[x * P + lane] = fmaf(eps * var[x], p[x * P + lane], q[x * P + lane]);
        }
      __syncthreads();
      const float h = (s + 1 == nfrog) ? 0.5f * eps : eps;
      for (int r = g; r < L; r += G)
        for (int c = 0; c < L; ++c) {
          const int x = r * L + c;
          p[x * P + lane] -= h * hmc_grad_u(cq, x, r, c, L, beta, m0sq, lam4);
        }
    }
    // H_new: kinetic, S_E (Eq. 1, forward neighbours), U0 over this warp's rows
    float K1 = 0.f, Sp = 0.f, Up = 0.f;
    for (int r = g; r < L; r += G) {
      const int rs = r + 1 == L ? 0 : r + 1;
      float rowS = 0.f, rowU = 0.f, rowK = 0.f;
      for (int c = 0; c < L; ++c) {
        const int x = r * L + c, ce = c + 1 == L ? 0 : c + 1;
        const float a = cq[x * P], b = cq[(r * L + ce) * P], d = cq[(rs * L + c) * P];
        const float e1 = b - a, e2 = d - a, a2 = a * a, pp = p[x * P + lane];
        rowS += 0.5f * (e1 * e1 + e2 * e2) + a2 * (0.5f * m0sq + lam * a2);
        rowU = fmaf(0.5f, a2, rowU);
        rowK = fmaf(0.5f * var[x] * pp, pp, rowK);
      }
      Sp += rowS; Up += rowU; K1 += rowK;
    }
    red[g * P + lane] = make_float4(K0, K1, Sp, Up);
    __syncthreads();
    if (g == 0) {
      float4 tot = make_float4(0.f, 0.f, 0.f, 0.f);
#pragma unroll
      for (int m = 0; m < G; ++m) {
        const float4 v = red[m * P + lane];
        tot.x += v.x; tot.y += v.y; tot.z += v.z; tot.w += v.w;
      }
      int acc = 0;
      if (live) {
        const float lu = log_uniform(seed, TAG_ACC, t, (uint32_t)i);
        // (H_old - H_new) - ln u with the differences taken term by term
        const float margin = ((Ui - tot.w) + beta * (Si - tot.z) + (tot.x - tot.y)) - lu;
        acc = margin > 0.f;
        if (acc) { Si = tot.z; Ui = tot.w; ++nacc; }
        if (acc_out) acc_out[(size_t)j * N + i] = (uint8_t)acc;
        if (margin_out) margin_out[(size_t)j * N + i] = margin;
      }
      flag[lane] = acc;
    }
    __syncthreads();
    if (flag[lane])
      for (int x = g; x < V; x += G) cur[x * P + lane] = q[x * P + lane];
    __syncthreads();
  }
  if (live) {
    for (int x = g; x < V; x += G) phi[(size_t)x * ld + i] = cur[x * P + lane];
    if (g == 0) { S[i] = Si; U0[i] = Ui; }
  }
  if (g == 0) {
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) nacc += __shfl_xor_sync(0xffffffffu, nacc, o);
    if (lane == 0 && nacc) atomicAdd(&ctrl->n_accept, nacc);
  }
}

static size_t hmc_smem_bytes(int V) {
  return ((size_t)3 * V * hm::P + 2 * V) * sizeof(float) + (size_t)hm::G * hm::P * sizeof(float4);
}

bool hmc_supported(int V) { return hmc_smem_bytes(V) <= 200 * 1024; }

void launch_hmc(float* phi, float* S, float* U0, const float* Sigma, int N, int ld, Model md,
                float eps, int nfrog, uint64_t seed, uint32_t t0, int k, Ctrl* ctrl,
                uint8_t* acc_out, float* margin_out, int respect_done, cudaStream_t st) {
  static bool attr_done = false;
  if (!attr_done) {
    cudaFuncSetAttribute(hmc_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, 200 * 1024);
    attr_done = true;
  }
  ++g_launches;
  hmc_kernel<<<(N + hm::P - 1) / hm::P, hm::THREADS, hmc_smem_bytes(md.V), st>>>(
      phi, S, U0, Sigma, N, ld, md, eps, nfrog, seed, t0, k, ctrl, acc_out, margin_out,
      respect_done);
}

}  // namespace phi4
