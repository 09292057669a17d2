// mutate_generic.cu -- M1-M4 for any lattice size, one launch triple per step:
//   normals_kernel   z[y][i]  (Philox, never reused across steps)
//   propose_kernel   phi'[x][i] = phi[x][i] + s * sum_{y<=x} Lc[x][y] z[y][i]   (FP32 SIMT GEMM)
//   accept_kernel    per-site action differences, Metropolis / constrained accept, commit
// This is the size-agnostic path (and the reference point for the fused tcgen05 kernel): its HBM
// traffic is per step, not per temperature.
#include "kernels.cuh"
#include "philox.cuh"

namespace phi4 {

__global__ void normals_kernel(float* __restrict__ Z, int N, int ld, int V, uint64_t seed,
                               uint32_t tag, uint32_t t, const Ctrl* ctrl, int respect_done) {
  if (respect_done && ctrl->done) return;
  int i = blockIdx.x * blockDim.x + threadIdx.x;
  int q = blockIdx.y;
  if (i >= ld) return;
  float z[4] = {0.f, 0.f, 0.f, 0.f};
  if (i < N) normals4(seed, tag, t, (uint32_t)i, (uint32_t)q, z);
#pragma unroll
  for (int j = 0; j < 4; ++j) {
    int x = 4 * q + j;
    if (x < V) Z[(size_t)x * ld + i] = z[j];
  }
}

// C[x][i] = phi[x][i] (or mu[x]) + s * sum_y Lc[x][y] Z[y][i].  64x64 tile, BK=16, 4x4 per thread.  Lc is
// lower-triangular, so the y loop of a tile ends at its last row.
__global__ void __launch_bounds__(256)
propose_kernel(const float* __restrict__ Lc, const float* __restrict__ Z,
               const float* __restrict__ phi, float* __restrict__ phip, int V, int ld, float s,
               const float* __restrict__ mu, int zero_base, const Ctrl* ctrl, int respect_done) {
  if (respect_done && ctrl->done) return;
  __shared__ float As[16][64 + 4];
  __shared__ __align__(16) float Bs[16][64];
  const int x0 = blockIdx.y * 64, i0 = blockIdx.x * 64;
  const int tx = threadIdx.x & 15, ty = threadIdx.x >> 4;
  // two-level accumulation (fold every 512 y's): fp32 rounding of the V-term sum ~ sqrt(512) +
  // sqrt(V/512) instead of sqrt(V), which keeps the V = 4096 margins inside the 1e-4 band
  float acc[4][4], tot[4][4];
#pragma unroll
  for (int a = 0; a < 4; ++a)
#pragma unroll
    for (int b = 0; b < 4; ++b) { acc[a][b] = 0.f; tot[a][b] = 0.f; }
  int since = 0;
  const int kend = min(V, x0 + 64);
  const int am = threadIdx.x >> 2, ak = (threadIdx.x & 3) * 4;  // A loader: row am, 4 k's
  const int bk = threadIdx.x >> 4, bn = (threadIdx.x & 15) * 4; // B loader: row bk, 4 i's
  for (int k0 = 0; k0 < kend; k0 += 16) {
#pragma unroll
    for (int j = 0; j < 4; ++j) {
      int x = x0 + am, y = k0 + ak + j;
      As[ak + j][am] = (x < V && y < V) ? Lc[(size_t)x * V + y] : 0.f;
    }
    {
      int y = k0 + bk;
      float4 v = make_float4(0.f, 0.f, 0.f, 0.f);
      if (y < V) v = *reinterpret_cast<const float4*>(Z + (size_t)y * ld + i0 + bn);
      *reinterpret_cast<float4*>(&Bs[bk][bn]) = v;
    }
    __syncthreads();
#pragma unroll
    for (int kk = 0; kk < 16; ++kk) {
      float a[4], b[4];
#pragma unroll
      for (int j = 0; j < 4; ++j) a[j] = As[kk][ty * 4 + j];
      float4 bv = *reinterpret_cast<const float4*>(&Bs[kk][tx * 4]);
      b[0] = bv.x; b[1] = bv.y; b[2] = bv.z; b[3] = bv.w;
#pragma unroll
      for (int p = 0; p < 4; ++p)
#pragma unroll
        for (int r = 0; r < 4; ++r) acc[p][r] = fmaf(a[p], b[r], acc[p][r]);
    }
    __syncthreads();
    if (++since == 32) {
      since = 0;
#pragma unroll
      for (int p = 0; p < 4; ++p)
#pragma unroll
        for (int r = 0; r < 4; ++r) { tot[p][r] += acc[p][r]; acc[p][r] = 0.f; }
    }
  }
#pragma unroll
  for (int p = 0; p < 4; ++p)
#pragma unroll
    for (int r = 0; r < 4; ++r) acc[p][r] += tot[p][r];
#pragma unroll
  for (int p = 0; p < 4; ++p) {
    int x = x0 + ty * 4 + p;
    if (x < V) {
      size_t o = (size_t)x * ld + i0 + tx * 4;
      // independent proposal (IRMH): the base point is the particle mean, not the particle
      // zero base (slice sampling): the output is the direction s * Lc z itself
      float4 f = zero_base ? make_float4(0.f, 0.f, 0.f, 0.f)
                 : mu      ? make_float4(mu[x], mu[x], mu[x], mu[x])
                           : *reinterpret_cast<const float4*>(phi + o);
      f.x = fmaf(s, acc[p][0], f.x);
      f.y = fmaf(s, acc[p][1], f.y);
      f.z = fmaf(s, acc[p][2], f.z);
      f.w = fmaf(s, acc[p][3], f.w);
      *reinterpret_cast<float4*>(phip + o) = f;
    }
  }
}

// Per-site differences of Eq. 1 and U0 between phi' and phi, written so that nothing cancels
// (SURVEY H3): with a = phi_x, b / c its forward neighbours and primes for the proposal,
//   d kin  = kappa/2 [(e'-e)(e'+e) + (f'-f)(f'+f)],  e = b-a, f = c-a   (hk = kappa/2; 1/2 for Eq. 1)
//   d mass + d quartic = (a'^2-a^2) (1/2 m0^2 + lambda (a'^2+a^2)),   dU0 = 1/2 (a'^2-a^2)
__device__ __forceinline__ void site_diff(float a, float b, float c, float a2, float b2, float c2,
                                          float hk, float hm, float lam, float& dS, float& dU) {
  float q = (a2 - a) * (a2 + a);
  float e = b - a, e2 = b2 - a2, f = c - a, f2 = c2 - a2;
  dS += hk * ((e2 - e) * (e2 + e) + (f2 - f) * (f2 + f)) + q * (hm + lam * (a2 * a2 + a * a));
  dU += 0.5f * q;
}

// Block = 32 particles x 8 row groups (one warp per group).  Phase 1: partial dS, dU0 over the
// group's lattice rows.  Phase 2: warp 0 decides (R4 margin; NS: also S' < S_star).  Phase 3:
// every group commits its rows of the accepted particles.
// G row groups (8, 16 or 32 warps): a small population does not fill the GPU with 8-warp blocks and
// a warp then walks a long band of rows with ~L2-latency per site; 32 groups shorten the band.
// NR > 0: column walk over bands of at most NR rows (large populations); NR = 0: row walk.
template <bool IRMH, int G, int NR>
__global__ void __launch_bounds__(32 * G)
accept_kernel(float* __restrict__ phi, const float* __restrict__ phip, float* __restrict__ S,
              float* __restrict__ U0, int N, int ld, Model md, int mode, uint64_t seed,
              uint32_t tag_acc, uint32_t t, Ctrl* ctrl, uint8_t* __restrict__ acc_out,
              float* __restrict__ margin_out, int respect_done, const float* __restrict__ Z,
              float* __restrict__ W2) {
  pdl_enter();
  if (respect_done && ctrl->done) return;
  __shared__ float ps[G][32], pu[G][32], pz[IRMH ? G : 1][32];
  __shared__ int flag[32];
  const int lane = threadIdx.x & 31, g = threadIdx.x >> 5;
  const int i = blockIdx.x * 32 + lane;
  const int L = md.L;
  const float hm = 0.5f * md.m0sq, lam = md.lam, hk = 0.5f * md.kappa;
  // each warp owns a contiguous band of lattice rows
  const int band = (L + G - 1) / G, r_lo = min(L, g * band), r_hi = min(L, r_lo + band);
  float dS = 0.f, dU = 0.f, z2 = 0.f;
  if (i < N) {
    if (IRMH) {                       // |z|^2 of this band: log q(phi') = -1/2 |z|^2 + const
      for (int x = r_lo * L; x < r_hi * L; ++x) {
        const float z = Z[(size_t)x * ld + i];
        z2 = fmaf(z, z, z2);
      }
    }
    if constexpr (NR > 0) {
      // Column walk (large populations; a small one is latency-bound and prefers the row walk):
      // the band's rows (<= NR) and the halo row below it are held in registers for the current
      // column and the two columns to its right, so every site of phi and phi' is loaded once
      // (plus the halo row and the wrap-around column) instead of once as a site and again as the
      // "down" neighbour of the row above.  The kernel is HBM-bound at C3 / C4 and the bytes in
      // flight are what its registers can hold: loads run two columns ahead of the arithmetic
      // (one column ahead with 8-row bands: 30-55 KB in flight per SM, 3.4-4.8 TB/s, round 1).
      const int nr = r_hi - r_lo;
      const int rh = (r_hi == L) ? 0 : r_hi;              // halo row below the band
      float A[NR + 1], A2[NR + 1], Bn[NR + 1], B2[NR + 1], Cn[NR + 1], C2[NR + 1], rS[NR], rU[NR];
#pragma unroll
      for (int q = 0; q < NR; ++q) { rS[q] = 0.f; rU[q] = 0.f; }
      auto load_col = [&](int c, float (&X)[NR + 1], float (&X2)[NR + 1]) {
#pragma unroll
        for (int q = 0; q < NR; ++q)
          if (q < nr) {
            const size_t o = ((size_t)(r_lo + q) * L + c) * ld + i;
            X[q] = phi[o]; X2[q] = phip[o];
          }
        const size_t o = ((size_t)rh * L + c) * ld + i;
        X[NR] = phi[o]; X2[NR] = phip[o];
      };
      if (nr > 0) {
        load_col(0, A, A2);
        load_col(1 % L, Bn, B2);
        for (int c = 0; c < L; ++c) {
          if (c + 2 <= L) load_col(c + 2 == L ? 0 : c + 2, Cn, C2);
#pragma unroll
          for (int q = 0; q < NR; ++q)
            if (q < nr) {
              const float d = (q + 1 < nr) ? A[q + 1 < NR ? q + 1 : NR] : A[NR];
              const float d2 = (q + 1 < nr) ? A2[q + 1 < NR ? q + 1 : NR] : A2[NR];
              site_diff(A[q], Bn[q], d, A2[q], B2[q], d2, hk, hm, lam, rS[q], rU[q]);
            }
#pragma unroll
          for (int q = 0; q <= NR; ++q) { A[q] = Bn[q]; A2[q] = B2[q]; Bn[q] = Cn[q]; B2[q] = C2[q]; }
        }
#pragma unroll
        for (int q = 0; q < NR; ++q)
          if (q < nr) { dS += rS[q]; dU += rU[q]; }
      }
    } else {
      // Row walk, CH columns at a time: the 4 CH loads of a chunk are issued before its arithmetic (a
      // small population is latency-bound: one column at a time paid an L2 / HBM round trip per site,
      // 14 us per step at N = 5000, L = 15).  Same order of additions as a plain column loop.
      constexpr int CH = 8;
      for (int r = r_lo; r < r_hi; ++r) {
        int rn = (r + 1 == L) ? 0 : r + 1;
        size_t ro = (size_t)r * L * ld + i, rno = (size_t)rn * L * ld + i;
        float a = phi[ro], a2 = phip[ro];
        float rS = 0.f, rU = 0.f;       // per-row partial sums: two-level fp32 accumulation
        for (int c0 = 0; c0 < L; c0 += CH) {
          float b[CH], b2[CH], d[CH], d2[CH];
#pragma unroll
          for (int u = 0; u < CH; ++u) {
            const int c = c0 + u;
            if (c < L) {
              const int cn = (c + 1 == L) ? 0 : c + 1;
              b[u] = phi[ro + (size_t)cn * ld]; b2[u] = phip[ro + (size_t)cn * ld];
              d[u] = phi[rno + (size_t)c * ld]; d2[u] = phip[rno + (size_t)c * ld];
            }
          }
#pragma unroll
          for (int u = 0; u < CH; ++u) {
            if (c0 + u < L) {
              site_diff(a, b[u], d[u], a2, b2[u], d2[u], hk, hm, lam, rS, rU);
              a = b[u];
              a2 = b2[u];
            }
          }
        }
        dS += rS;
        dU += rU;
      }
    }
  }
  ps[g][lane] = dS;
  pu[g][lane] = dU;
  if (IRMH) pz[g][lane] = z2;
  __syncthreads();
  if (g == 0) {
    int acc = 0;
    if (i < N) {
      float tS = 0.f, tU = 0.f;
#pragma unroll
      for (int m = 0; m < G; ++m) { tS += ps[m][lane]; tU += pu[m][lane]; }
      float lu = log_uniform(seed, tag_acc, t, (uint32_t)i);
      float Si = S[i], margin;
      if (!IRMH && mode == MODE_SMC) {
        margin = -(tU + (float)ctrl->beta * tS) - lu;
        acc = margin > 0.f;
      } else if (IRMH) {
        float tZ = 0.f;
#pragma unroll
        for (int m = 0; m < G; ++m) tZ += pz[m][lane];
        // log q(phi) - log q(phi') = 1/2 |z|^2 - 1/2 |w|^2, w = Lc^-1 (phi - mu) (reading A15)
        margin = -(tU + (float)ctrl->beta * tS) + 0.5f * (tZ - W2[i]) - lu;
        acc = margin > 0.f;
        if (acc) W2[i] = tZ;
      } else {
        margin = -tU - lu;
        acc = (margin > 0.f) && (Si + tS < (float)ctrl->S_star);
      }
      if (acc) {
        S[i] = Si + tS;
        U0[i] += tU;
      }
      if (acc_out) acc_out[i] = (uint8_t)acc;
      if (margin_out) margin_out[i] = margin;
    }
    flag[lane] = acc;
    unsigned m = __ballot_sync(0xffffffffu, acc);
    if (lane == 0 && m) atomicAdd(&ctrl->n_accept, (unsigned)__popc(m));
  }
  __syncthreads();
  if (i < N && flag[lane]) {
    for (int r = r_lo; r < r_hi; ++r) {
      size_t ro = (size_t)r * L * ld + i;
      if constexpr (NR == 0) {                 // (latency-bound sizes: eight loads in flight per thread)
        for (int c0 = 0; c0 < L; c0 += 8) {
          float v[8];
#pragma unroll
          for (int u = 0; u < 8; ++u) if (c0 + u < L) v[u] = phip[ro + (size_t)(c0 + u) * ld];
#pragma unroll
          for (int u = 0; u < 8; ++u) if (c0 + u < L) phi[ro + (size_t)(c0 + u) * ld] = v[u];
        }
      } else {
        for (int c = 0; c < L; ++c) phi[ro + (size_t)c * ld] = phip[ro + (size_t)c * ld];
      }
    }
  }
}

// M3 + M4 of step j (step counter a.t0 + j): action differences between a.phip and a.phi,
// decision, commit.
void launch_accept_step(const MutateArgs& a, int j, cudaStream_t st) {
  const uint32_t t = a.t0 + (uint32_t)j;
  // fewer than two 8-warp blocks per SM and more than 8 lattice rows: one warp per row instead
  const bool wide = a.md.L > 8 && a.ld / 32 < 2 * 148;
  // large populations: column walk over bands of <= 4 lattice rows (8, 16 or 32 row groups)
  const bool colwalk = !wide && a.ld >= 8192 && a.md.L >= 25 && a.md.L <= 128;
  ++g_launches;
  auto launch_accept = [&](auto kern, int G) {
    launch_pdl(kern, a.ld / 32, 32 * G, 0, st,
               a.phi, a.phip, a.S, a.U0, a.N, a.ld, a.md, a.mode, a.seed, a.tag_acc, t, a.ctrl,
               a.acc_out ? a.acc_out + (size_t)j * a.N : nullptr,
               a.margin_out ? a.margin_out + (size_t)j * a.N : nullptr, a.respect_done,
               (const float*)nullptr, (float*)nullptr);
  };
  if (wide) launch_accept(accept_kernel<false, 32, 0>, 32);
  else if (colwalk && a.md.L <= 32) launch_accept(accept_kernel<false, 8, 4>, 8);
  else if (colwalk && a.md.L <= 64) launch_accept(accept_kernel<false, 16, 4>, 16);
  else if (colwalk) launch_accept(accept_kernel<false, 32, 4>, 32);
  else launch_accept(accept_kernel<false, 8, 0>, 8);
}

// Lsplit != nullptr selects the tcgen05 proposal (propose_tc.cu) for M1 + M2; a.Z must then hold
// 2 V ld floats.  The accept / commit step is the same either way.
void launch_mutate_generic(const MutateArgs& a, float* Lsplit, cudaStream_t st) {
  const int V = a.md.V;
  dim3 gz((a.ld + 127) / 128, (V + 3) / 4);
  dim3 gp(a.ld / 64, (V + 63) / 64);
  if (Lsplit) {
    launch_propose_lsplit(a.Lc, V, a.ld, a.s, Lsplit, a.ctrl, a.respect_done, st, a.tc_f16);
  }
  // Normals of step j+1 while the GEMM of step j runs (they depend on nothing but the counters):
  // drawn by two spare warps inside every GEMM CTA into the other buffer.  (Round 2 first launched
  // them as a kernel of their own on a side stream: beside a persistent GEMM CTA -- 12 warps' worth
  // of registers -- no block of another kernel fits, so they only started when GEMM CTAs exited and
  // then ran against the accept kernel: C3 0.55 ms per step for 0.23 + 0.16 ms of GEMM + accept.)
  // Only where a CTA's GEMM work is long enough to hide its share of the normals.
  const bool fuse = Lsplit && a.Z2 && a.k > 1 && (size_t)a.ld * V >= ((size_t)1 << 22);
  float* zbuf[2] = {a.Z, fuse ? a.Z2 : a.Z};
  // small populations: the normals of a batch of steps per launch (one step alone is a launch-latency-sized
  // kernel: 4.5 us at N = 5000, L = 15 for 1.7 us of work)
  const int zb = (Lsplit && !fuse) ? propose_tc_zbatch(V, a.ld, a.tc_f16) : 1;
  const size_t zstep = Lsplit ? propose_tc_zstep_floats(V, a.ld, a.tc_f16) : 0;
  if (Lsplit && fuse)
    launch_normals_split(zbuf[0], a.N, a.ld, V, a.seed, a.tag_prop, a.t0, a.ctrl, a.respect_done, st, a.tc_f16);
  for (int j = 0; j < a.k; ++j) {
    uint32_t t = a.t0 + (uint32_t)j;
    if (Lsplit) {
      if (!fuse && j % zb == 0)
        launch_normals_split(zbuf[0], a.N, a.ld, V, a.seed, a.tag_prop, t, a.ctrl, a.respect_done, st, a.tc_f16,
                             a.k - j < zb ? a.k - j : zb);
      const NextNormals nx = {zbuf[(j + 1) & 1], a.N, a.seed, a.tag_prop, t + 1};
      launch_propose_tc(a.phi, a.phip, fuse ? zbuf[j & 1] : zbuf[0] + (size_t)(j % zb) * zstep, Lsplit, a.ld, V,
                        a.ctrl, a.respect_done, st, a.tc_f16, (fuse && j + 1 < a.k) ? &nx : nullptr);
    } else {
      ++g_launches; normals_kernel<<<gz, 128, 0, st>>>(a.Z, a.N, a.ld, V, a.seed, a.tag_prop, t, a.ctrl,
                                         a.respect_done);
      ++g_launches; propose_kernel<<<gp, 256, 0, st>>>(a.Lc, a.Z, a.phi, a.phip, V, a.ld, a.s, nullptr,
                                         0, a.ctrl, a.respect_done);
    }
    launch_accept_step(a, j, st);
  }
}

// ---------------------------------------------------------------------------------------------
// NEXT row f2: independent Metropolis-Hastings from the fitted Gaussian N(mu, Lc Lc^T)
// (PAPER.md:53(ii), :200; reading A15).  whiten_kernel: W2[i] = |Lc^-1 (phi_i - mu)|^2 by forward
// substitution, one warp per 32 particles, w in shared memory; FP64 accumulation (once per
// temperature: the solve amplifies rounding by cond(Lc), and W2 enters every margin).
// V <= 128.  FP64 accumulation (the solve amplifies rounding by cond(Lc) and W2 enters every margin).
// One thread per particle is a single dependent chain per SM sub-partition (16384 particles are 512
// warps on 592 sub-partitions): 111 us at C1.  Here a block is WH_P particles x 4 row lanes (256
// threads): thread (p, j) carries row x0 + j of the current 4-row block for particle p -- four
// independent FP64 chains over the column phases -- and the j = 0 threads then finish the 4 x 4
// diagonal block serially; two block barriers per row block.  The factor sits in shared memory as
// FP32 (rows padded to a multiple of four, zeros beyond the row end) and is read as broadcasts.
constexpr int WH_P = 64;
__host__ __device__ inline int wh_vp(int V) { return (V + 3) & ~3; }
__host__ __device__ inline size_t whiten_smem(int V) {
  return (size_t)wh_vp(V) * wh_vp(V) * sizeof(float) + ((size_t)V * WH_P + wh_vp(V)) * sizeof(double);
}
__global__ void __launch_bounds__(4 * WH_P)
whiten_small_kernel(const float* __restrict__ phi, const float* __restrict__ mu,
                    const float* __restrict__ Lc, float* __restrict__ W2, int N, int ld, int V,
                    const Ctrl* ctrl, int respect_done) {
  if (respect_done && ctrl->done) return;
  extern __shared__ double whd[];
  __shared__ double accs[3][WH_P];                              // row sums of rows x0 + 1 .. x0 + 3
  const int Vp = wh_vp(V);
  double* wsm = whd;                                            // [V][WH_P]
  double* invd = wsm + (size_t)V * WH_P;                        // [Vp] 1 / L_xx
  float* Lf = reinterpret_cast<float*>(invd + Vp);              // [Vp][Vp], zero outside the lower triangle
  const int tid = threadIdx.x, p = tid & (WH_P - 1), j = tid >> 6;   // j is warp-uniform
  const int i = blockIdx.x * WH_P + p;
  const bool live = i < N;
  // eight loads in flight per thread (the factor comes from L2: one round trip per batch)
  for (int e0 = 0; e0 < Vp * Vp; e0 += 8 * 4 * WH_P) {
    float v[8];
#pragma unroll
    for (int u = 0; u < 8; ++u) {
      const int e = e0 + u * 4 * WH_P + tid, x = e / Vp, y = e - x * Vp;
      v[u] = (x < V && y <= x) ? Lc[(size_t)x * V + y] : 0.f;
    }
#pragma unroll
    for (int u = 0; u < 8; ++u) {
      const int e = e0 + u * 4 * WH_P + tid;
      if (e < Vp * Vp) Lf[e] = v[u];
    }
  }
  for (int x = tid; x < Vp; x += 4 * WH_P) invd[x] = x < V ? 1.0 / (double)Lc[(size_t)x * V + x] : 0.0;
  __syncthreads();
  double w2 = 0.0;
  for (int x0 = 0; x0 < V; x0 += 4) {
    // the j = 0 threads need this row block's right-hand sides after the product loop
    double rhs[4];
    if (j == 0) {
#pragma unroll
      for (int m = 0; m < 4; ++m) {
        const int x = min(x0 + m, V - 1);
        rhs[m] = live ? (double)phi[(size_t)x * ld + i] - (double)mu[x] : 0.0;
      }
    }
    const float* row = Lf + (size_t)(x0 + j) * Vp;
    double a0 = 0.0, a1 = 0.0, a2 = 0.0, a3 = 0.0;
    for (int y = 0; y < x0; y += 4) {          // x0 is a multiple of 4
      const float4 l = *reinterpret_cast<const float4*>(row + y);
      a0 = fma((double)l.x, wsm[y * WH_P + p], a0);
      a1 = fma((double)l.y, wsm[(y + 1) * WH_P + p], a1);
      a2 = fma((double)l.z, wsm[(y + 2) * WH_P + p], a2);
      a3 = fma((double)l.w, wsm[(y + 3) * WH_P + p], a3);
    }
    const double acc = (a0 + a1) + (a2 + a3);
    if (j > 0) accs[j - 1][p] = acc;
    __syncthreads();
    if (j == 0) {
      double wl[4];
#pragma unroll
      for (int m = 0; m < 4; ++m) {
        const int x = x0 + m;
        if (x < V) {
          double s = m > 0 ? accs[m - 1][p] : acc;
          const float* rm = Lf + (size_t)x * Vp + x0;
#pragma unroll
          for (int q = 0; q < 4; ++q)
            if (q < m) s = fma((double)rm[q], wl[q], s);
          const double v = (rhs[m] - s) * invd[x];
          wl[m] = v;
          wsm[x * WH_P + p] = v;
          w2 = fma(v, v, w2);
        }
      }
    }
    __syncthreads();
  }
  if (j == 0 && live) W2[i] = (float)w2;
}

// Any V <= 800: one warp per 32 particles, the factor read through the read-only cache.
__global__ void __launch_bounds__(32)
whiten_kernel(const float* __restrict__ phi, const float* __restrict__ mu,
              const float* __restrict__ Lc, float* __restrict__ W2, int N, int ld, int V,
              const Ctrl* ctrl, int respect_done) {
  if (respect_done && ctrl->done) return;
  extern __shared__ double wsm[];          // [V][32] w, then [V] 1 / L_xx
  double* invd = wsm + (size_t)V * 32;
  const int lane = threadIdx.x, i = blockIdx.x * 32 + lane;
  for (int x = lane; x < V; x += 32) invd[x] = 1.0 / (double)Lc[(size_t)x * V + x];
  __syncwarp();
  if (i >= N) return;
  double w2 = 0.0;
  for (int x0 = 0; x0 < V; x0 += 4) {
    const int nb = min(4, V - x0);
    const float* r0 = Lc + (size_t)x0 * V;
    const float* r1 = Lc + (size_t)min(x0 + 1, V - 1) * V;
    const float* r2 = Lc + (size_t)min(x0 + 2, V - 1) * V;
    const float* r3 = Lc + (size_t)min(x0 + 3, V - 1) * V;
    double a0 = 0.0, a1 = 0.0, a2 = 0.0, a3 = 0.0, c0 = 0.0, c1 = 0.0, c2 = 0.0, c3 = 0.0;
    for (int y = 0; y < x0; y += 2) {        // x0 is a multiple of 4: whole pairs
      const double w0 = wsm[y * 32 + lane], w1 = wsm[(y + 1) * 32 + lane];
      a0 = fma((double)__ldg(r0 + y), w0, a0); c0 = fma((double)__ldg(r0 + y + 1), w1, c0);
      a1 = fma((double)__ldg(r1 + y), w0, a1); c1 = fma((double)__ldg(r1 + y + 1), w1, c1);
      a2 = fma((double)__ldg(r2 + y), w0, a2); c2 = fma((double)__ldg(r2 + y + 1), w1, c2);
      a3 = fma((double)__ldg(r3 + y), w0, a3); c3 = fma((double)__ldg(r3 + y + 1), w1, c3);
    }
    const double acc[4] = {a0 + c0, a1 + c1, a2 + c2, a3 + c3};
    const float* rows[4] = {r0, r1, r2, r3};
    double wl[4];
#pragma unroll
    for (int j = 0; j < 4; ++j)
      if (j < nb) {
        const int x = x0 + j;
        double v = (double)phi[(size_t)x * ld + i] - (double)mu[x] - acc[j];
#pragma unroll
        for (int m = 0; m < 4; ++m)
          if (m < j) v -= (double)__ldg(rows[j] + x0 + m) * wl[m];
        v *= invd[x];
        wl[j] = v;
        wsm[x * 32 + lane] = v;
        w2 = fma(v, v, w2);
      }
  }
  W2[i] = (float)w2;
}

bool irmh_supported(int V) { return V >= 1 && V <= 800; }     // w [V][32] + 1 / L_xx [V] in FP64: 211 KB

void launch_mutate_irmh(const MutateArgs& a, const float* mu, float* W2, float* Lsplit, cudaStream_t st) {
  const int V = a.md.V;
  static bool attr_done = false;
  if (!attr_done) {
    cudaFuncSetAttribute(whiten_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, 800 * 33 * (int)sizeof(double));
    cudaFuncSetAttribute(whiten_small_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, 224 * 1024);
    attr_done = true;
  }
  ++g_launches;
  if (whiten_smem(V) <= (size_t)224 * 1024)
    whiten_small_kernel<<<(a.N + WH_P - 1) / WH_P, 4 * WH_P, whiten_smem(V), st>>>(
        a.phi, mu, a.Lc, W2, a.N, a.ld, V, a.ctrl, a.respect_done);
  else
    whiten_kernel<<<(a.N + 31) / 32, 32, (size_t)V * 33 * sizeof(double), st>>>(
        a.phi, mu, a.Lc, W2, a.N, a.ld, V, a.ctrl, a.respect_done);
  if (Lsplit) {                      // the k steps in the fused tcgen05 kernel
    launch_mutate_tc(a, Lsplit, st, mu, W2);
    return;
  }
  dim3 gz((a.ld + 127) / 128, (V + 3) / 4);
  dim3 gp(a.ld / 64, (V + 63) / 64);
  for (int j = 0; j < a.k; ++j) {
    uint32_t t = a.t0 + (uint32_t)j;
    ++g_launches; normals_kernel<<<gz, 128, 0, st>>>(a.Z, a.N, a.ld, V, a.seed, a.tag_prop, t, a.ctrl,
                                       a.respect_done);
    ++g_launches; propose_kernel<<<gp, 256, 0, st>>>(a.Lc, a.Z, a.phi, a.phip, V, a.ld, 1.0f, mu,
                                       0, a.ctrl, a.respect_done);
    ++g_launches; accept_kernel<true, 8, 0><<<a.ld / 32, 256, 0, st>>>(
        a.phi, a.phip, a.S, a.U0, a.N, a.ld, a.md, MODE_IRMH, a.seed, a.tag_acc, t, a.ctrl,
        a.acc_out ? a.acc_out + (size_t)j * a.N : nullptr,
        a.margin_out ? a.margin_out + (size_t)j * a.N : nullptr, a.respect_done, a.Z, W2);
  }
}

// ---------------------------------------------------------------------------------------------
// NEXT row f3: the slice-sampling inner kernel of nested sampling (PAPER.md:53(iv), :174; reading
// A16).  Per step: normals_kernel, propose_kernel with a zero base (d = Lc z), slice_kernel.
// Along the line phi + t d both S_E and U0 are polynomials in t (quartic / quadratic) whose
// coefficients are eight lattice sums; every Inside(t) test of the stepping-out and shrinkage
// loops is then O(1):
//   U0(t)  = U0 + t A1 + t^2 A2/2,                      A1 = sum f d, A2 = sum d^2
//   S_E(t) = S_E + t (K1 + m0^2 A1 + 4 lam Q1) + t^2 (K2/2 + m0^2 A2/2 + 6 lam Q2)
//                + t^3 4 lam Q3 + t^4 lam Q4,
//   K1 = sum_bonds (Df)(Dd), K2 = sum_bonds (Dd)^2, Q1..Q4 = sum f^3 d, f^2 d^2, f d^3, d^4.
// Block = 32 walkers x 8 row groups: partial sums per group, warp 0 runs the (divergent) scalar
// loops, every group then moves its rows of the walkers that found a point.
__global__ void __launch_bounds__(256)
slice_kernel(float* __restrict__ phi, const float* __restrict__ dir, float* __restrict__ S,
             float* __restrict__ U0, int N, int ld, Model md, float width, int m_expand,
             int max_shrink, uint64_t seed, uint32_t t, Ctrl* ctrl, int respect_done) {
  if (respect_done && ctrl->done) return;
  __shared__ float part[8][8][32];
  __shared__ float tsel[32];
  const int lane = threadIdx.x & 31, g = threadIdx.x >> 5;
  const int i = blockIdx.x * 32 + lane;
  const int L = md.L;
  const int band = (L + 7) >> 3, r_lo = g * band, r_hi = min(L, r_lo + band);
  float acc[8] = {0.f, 0.f, 0.f, 0.f, 0.f, 0.f, 0.f, 0.f};
  if (i < N) {
    for (int r = r_lo; r < r_hi; ++r) {
      const int rn = (r + 1 == L) ? 0 : r + 1;
      const size_t ro = (size_t)r * L * ld + i, rno = (size_t)rn * L * ld + i;
      float row[8] = {0.f, 0.f, 0.f, 0.f, 0.f, 0.f, 0.f, 0.f};   // two-level fp32 accumulation
      float f = phi[ro], d = dir[ro];
      for (int c = 0; c < L; ++c) {
        const int cn = (c + 1 == L) ? 0 : c + 1;
        const float fe = phi[ro + (size_t)cn * ld], de = dir[ro + (size_t)cn * ld];
        const float fs = phi[rno + (size_t)c * ld], ds = dir[rno + (size_t)c * ld];
        const float dfe = fe - f, dde = de - d, dfs = fs - f, dds = ds - d;
        const float f2 = f * f, d2 = d * d;
        row[0] = fmaf(f, d, row[0]);
        row[1] += d2;
        row[2] += dfe * dde + dfs * dds;
        row[3] += dde * dde + dds * dds;
        row[4] = fmaf(f2 * f, d, row[4]);
        row[5] = fmaf(f2, d2, row[5]);
        row[6] = fmaf(f * d, d2, row[6]);
        row[7] = fmaf(d2, d2, row[7]);
        f = fe;
        d = de;
      }
#pragma unroll
      for (int q = 0; q < 8; ++q) acc[q] += row[q];
    }
  }
#pragma unroll
  for (int q = 0; q < 8; ++q) part[q][g][lane] = acc[q];
  __syncthreads();
  if (g == 0) {
    float tacc = 0.f;
    if (i < N) {
      float v[8];
#pragma unroll
      for (int q = 0; q < 8; ++q) {
        float a = 0.f;
#pragma unroll
        for (int m = 0; m < 8; ++m) a += part[q][m][lane];
        v[q] = a;
      }
      const float lam = md.lam, m0 = md.m0sq;
      const float c1 = md.kappa * v[2] + m0 * v[0] + 4.f * lam * v[4];
      const float c2 = 0.5f * md.kappa * v[3] + 0.5f * m0 * v[1] + 6.f * lam * v[5];
      const float c3 = 4.f * lam * v[6], c4 = lam * v[7];
      const float u1 = v[0], u2 = 0.5f * v[1];
      const float S0 = S[i], Ub = U0[i], S_star = (float)ctrl->S_star;
      U4 w = philox_draw(seed, TAG_NS_SLICE, t, (uint32_t)i, 0u);
      const float u_h = (float)((w.x >> 8) + 1u) * 5.9604644775390625e-8f;
      const float u_b = (float)(w.y >> 8) * 5.9604644775390625e-8f;
      const float u_j = (float)(w.z >> 8) * 5.9604644775390625e-8f;
      const float logy = -Ub + logf(u_h);
      float Sx = S0, Ux = Ub;
      auto inside = [&](float tt) {
        Sx = fmaf(tt, fmaf(tt, fmaf(tt, fmaf(tt, c4, c3), c2), c1), S0);
        Ux = fmaf(tt, fmaf(tt, u2, u1), Ub);
        return Sx < S_star && -Ux > logy;
      };
      float l = -width * u_b, r = l + width;
      int J = (int)floorf((float)m_expand * u_j), K = m_expand - 1 - J;
      while (J > 0 && inside(l)) { l -= width; --J; }
      while (K > 0 && inside(r)) { r += width; --K; }
      for (int m = 0; m < max_shrink; ++m) {
        if ((m & 3) == 0) w = philox_draw(seed, TAG_NS_SLICE, t, (uint32_t)i, 1u + (uint32_t)(m >> 2));
        const uint32_t wd = (m & 3) == 0 ? w.x : (m & 3) == 1 ? w.y : (m & 3) == 2 ? w.z : w.w;
        const float u = ((float)(wd >> 8) + 0.5f) * 5.9604644775390625e-8f;
        const float tt = fmaf(u, r - l, l);
        if (inside(tt)) {
          tacc = tt;
          S[i] = Sx;
          U0[i] = Ux;
          break;
        }
        if (tt < 0.f) l = tt; else r = tt;
      }
    }
    tsel[lane] = tacc;
    const unsigned moved = __ballot_sync(0xffffffffu, tacc != 0.f);
    if (lane == 0 && moved) atomicAdd(&ctrl->n_accept, (unsigned)__popc(moved));
  }
  __syncthreads();
  const float tt = tsel[lane];
  if (i < N && tt != 0.f) {
    for (int r = r_lo; r < r_hi; ++r) {
      const size_t ro = (size_t)r * L * ld + i;
      for (int c = 0; c < L; ++c) {
        const size_t o = ro + (size_t)c * ld;
        phi[o] = fmaf(tt, dir[o], phi[o]);
      }
    }
  }
}

// a.phip receives the direction; a.mode / a.s / acc_out / margin_out are unused
void launch_ns_slice(const MutateArgs& a, float width, int m_expand, int max_shrink, cudaStream_t st) {
  const int V = a.md.V;
  dim3 gz((a.ld + 127) / 128, (V + 3) / 4);
  dim3 gp(a.ld / 64, (V + 63) / 64);
  for (int j = 0; j < a.k; ++j) {
    const uint32_t t = a.t0 + (uint32_t)j;
    ++g_launches; normals_kernel<<<gz, 128, 0, st>>>(a.Z, a.N, a.ld, V, a.seed, TAG_NS_PROP, t, a.ctrl,
                                       a.respect_done);
    ++g_launches; propose_kernel<<<gp, 256, 0, st>>>(a.Lc, a.Z, a.phi, a.phip, V, a.ld, 1.0f, nullptr, 1,
                                       a.ctrl, a.respect_done);
    ++g_launches; slice_kernel<<<a.ld / 32, 256, 0, st>>>(a.phi, a.phip, a.S, a.U0, a.N, a.ld, a.md, width,
                                     m_expand, max_shrink, a.seed, t, a.ctrl, a.respect_done);
  }
}

}  // namespace phi4
