// covchol.cu -- C1 (particle covariance) and C2 (Cholesky), readings A4 / R6.
//   mu_x = (1/N) sum_i phi[x][i];  Sigma = (1/(N-1)) sum_i (phi_i - mu)(phi_i - mu)^T
//   Sigma (+ jitter on retry) = Lc Lc^T, Lc lower-triangular, strict upper = 0.
// FP32 SIMT version: 64x64 "NT" tiles (both operands contiguous along the contraction index),
// lower-triangular tiles only, deterministic split-K for small V.  One CTA factorises V <= 160 in
// shared memory; larger V use a blocked right-looking factorisation (64-wide panels: diagonal
// block, row solves, trailing update with the same NT tile).
#include "kernels.cuh"

namespace phi4 {

// AMAX: also amax[x] = max_i |phi[x][i]| + |mu[x]| >= max_i |phi[x][i] - mu[x]| (the scale of the FP16
// covariance operands, syrk_tc.cu)
template <bool AMAX>
__global__ void __launch_bounds__(256)
mean_kernel(const float* __restrict__ phi, int N, int ld, float* __restrict__ mu,
            float* __restrict__ amax, const Ctrl* ctrl, int respect_done) {
  pdl_enter();
  __shared__ double scratch[33];
  if (respect_done && ctrl->done) return;
  float big = 0.f;
  const float* row = phi + (size_t)blockIdx.x * ld;
  // ld is a multiple of 128 and pad particles hold zeros: whole float4s.  Two-level sums: at most 32
  // terms in FP32 (four partial sums of eight), folded into FP64 -- one conversion and one FP64 add per
  // 32 terms instead of per term (half of this latency-sized kernel's instructions at C1)
  double a = 0.0;
  const float4* row4 = reinterpret_cast<const float4*>(row);
  const int n4 = ld / 4, stride = blockDim.x;
  for (int i0 = threadIdx.x; i0 < n4; i0 += 8 * stride) {
    float f0 = 0.f, f1 = 0.f, f2 = 0.f, f3 = 0.f;
#pragma unroll
    for (int u = 0; u < 8; ++u) {
      const int i = i0 + u * stride;
      if (i < n4) {
        const float4 v = row4[i];
        f0 += v.x; f1 += v.y; f2 += v.z; f3 += v.w;
        if (AMAX) big = fmaxf(fmaxf(big, fmaxf(fabsf(v.x), fabsf(v.y))), fmaxf(fabsf(v.z), fabsf(v.w)));
      }
    }
    a += (double)((f0 + f1) + (f2 + f3));
  }
  a = block_sum(a, scratch);
  if (threadIdx.x == 0) mu[blockIdx.x] = (float)(a / (double)N);
  if (AMAX) {
    __shared__ float bigs[8];
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) big = fmaxf(big, __shfl_xor_sync(0xffffffffu, big, o));
    if ((threadIdx.x & 31) == 0) bigs[threadIdx.x >> 5] = big;
    __syncthreads();
    if (threadIdx.x == 0) {
      for (int w = 1; w < 8; ++w) big = fmaxf(big, bigs[w]);
      amax[blockIdx.x] = big + fabsf((float)(a / (double)N));
    }
  }
}

// acc[p][r] += sum_{k in [kb,ke)} (A[(x0+ty*4+p)*lda + k] - mx) (A[(y0+tx*4+r)*lda + k] - my)
// Rows >= M and columns k >= kvalid contribute zero.  VEC: lda % 4 == 0 and kb % 16 == 0.
template <bool VEC>
__device__ __forceinline__ void nt_tile(const float* __restrict__ A, size_t lda, int x0, int y0,
                                        int M, int kb, int ke, int kvalid,
                                        const float* __restrict__ mu, float (&acc)[4][4],
                                        float (&As)[16][68], float (&Bs)[16][68]) {
  const int tx = threadIdx.x & 15, ty = threadIdx.x >> 4;
  const int lr = threadIdx.x >> 2, lk = (threadIdx.x & 3) * 4;
  const int xr = x0 + lr, yr = y0 + lr;
  const float mx = (mu && xr < M) ? mu[xr] : 0.f;
  const float my = (mu && yr < M) ? mu[yr] : 0.f;
  // Two-level accumulation: `acc` runs over 1024 contraction indices at a time and is then folded
  // into `tot`, so the fp32 rounding grows like sqrt(1024) + sqrt(K/1024) instead of sqrt(K)
  // (K = N = 131072 particles at C4 would otherwise miss the 1e-5 covariance tolerance).
  float tot[4][4];
#pragma unroll
  for (int p = 0; p < 4; ++p)
#pragma unroll
    for (int r = 0; r < 4; ++r) { tot[p][r] = acc[p][r]; acc[p][r] = 0.f; }
  int since = 0;
  // the global loads of slab k0 + 16 are issued before the FMAs of slab k0 (register double
  // buffer): their latency hides behind the 256 FMAs per thread instead of stalling every slab
  float va[4], vb[4];
  auto load_slab = [&](int k0) {
    if (VEC) {
      float4 a4 = make_float4(0.f, 0.f, 0.f, 0.f), b4 = a4;
      if (xr < M) a4 = *reinterpret_cast<const float4*>(A + (size_t)xr * lda + k0 + lk);
      if (yr < M) b4 = *reinterpret_cast<const float4*>(A + (size_t)yr * lda + k0 + lk);
      va[0] = a4.x; va[1] = a4.y; va[2] = a4.z; va[3] = a4.w;
      vb[0] = b4.x; vb[1] = b4.y; vb[2] = b4.z; vb[3] = b4.w;
    } else {
#pragma unroll
      for (int j = 0; j < 4; ++j) {
        int k = k0 + lk + j;
        va[j] = (xr < M && k < ke) ? A[(size_t)xr * lda + k] : 0.f;
        vb[j] = (yr < M && k < ke) ? A[(size_t)yr * lda + k] : 0.f;
      }
    }
  };
  if (kb < ke) load_slab(kb);
  for (int k0 = kb; k0 < ke; k0 += 16) {
#pragma unroll
    for (int j = 0; j < 4; ++j) {
      int k = k0 + lk + j;
      bool ok = k < kvalid && k < ke;
      As[lk + j][lr] = (ok && xr < M) ? va[j] - mx : 0.f;
      Bs[lk + j][lr] = (ok && yr < M) ? vb[j] - my : 0.f;
    }
    __syncthreads();
    if (k0 + 16 < ke) load_slab(k0 + 16);
#pragma unroll
    for (int kk = 0; kk < 16; ++kk) {
      const float4 a4 = *reinterpret_cast<const float4*>(&As[kk][ty * 4]);
      const float4 b4 = *reinterpret_cast<const float4*>(&Bs[kk][tx * 4]);
      const float a[4] = {a4.x, a4.y, a4.z, a4.w}, b[4] = {b4.x, b4.y, b4.z, b4.w};
#pragma unroll
      for (int p = 0; p < 4; ++p)
#pragma unroll
        for (int r = 0; r < 4; ++r) acc[p][r] = fmaf(a[p], b[r], acc[p][r]);
    }
    __syncthreads();
    if (++since == 64) {
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
}

// linear index t -> lower-triangular tile (tr, tc), tc <= tr
__device__ __forceinline__ void tri_tile(int t, int& tr, int& tc) {
  tr = (int)((sqrtf(8.f * (float)t + 1.f) - 1.f) * 0.5f);
  while ((tr + 1) * (tr + 2) / 2 <= t) ++tr;
  while (tr * (tr + 1) / 2 > t) --tr;
  tc = t - tr * (tr + 1) / 2;
}

// Split-K partial covariance sums: partial[z][x][y] over the particle chunk z.
__global__ void __launch_bounds__(256)
syrk_partial_kernel(const float* __restrict__ phi, int N, int ld, int V,
                    const float* __restrict__ mu, float* __restrict__ partial, int chunk,
                    const Ctrl* ctrl, int respect_done) {
  pdl_enter();
  if (respect_done && ctrl->done) return;
  __shared__ __align__(16) float As[16][68], Bs[16][68];
  int tr, tc;
  tri_tile(blockIdx.x, tr, tc);
  const int x0 = tr * 64, y0 = tc * 64;
  const int kb = blockIdx.y * chunk, ke = min(ld, kb + chunk);
  float acc[4][4];
#pragma unroll
  for (int p = 0; p < 4; ++p)
#pragma unroll
    for (int r = 0; r < 4; ++r) acc[p][r] = 0.f;
  nt_tile<true>(phi, (size_t)ld, x0, y0, V, kb, ke, N, mu, acc, As, Bs);
  const int tx = threadIdx.x & 15, ty = threadIdx.x >> 4;
  float* out = partial + (size_t)blockIdx.y * V * V;
#pragma unroll
  for (int p = 0; p < 4; ++p)
#pragma unroll
    for (int r = 0; r < 4; ++r) {
      int x = x0 + ty * 4 + p, y = y0 + tx * 4 + r;
      if (x < V && y < V) out[(size_t)x * V + y] = acc[p][r];
    }
}

// Sigma[x][y] = Sigma[y][x] = (sum_z partial[z][x][y]) / (N-1) for y <= x, fixed summation order.
// LANES = 8 (small V: few entries, many splits): eight lanes per entry each sum every eighth split,
// then a fixed shuffle tree.  LANES = 1 (large V): one thread per entry, coalesced along y.
template <int LANES>
__global__ void syrk_reduce_kernel(const float* __restrict__ partial, int nsplit, int V, int N,
                                   float* __restrict__ Sigma, const Ctrl* ctrl, int respect_done) {
  pdl_enter();
  if (respect_done && ctrl->done) return;
  const size_t t = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
  const size_t idx = t / LANES;
  const int part = (int)(t % LANES);
  const bool in = idx < (size_t)V * V;
  const int x = in ? (int)(idx / V) : 0, y = in ? (int)(idx - (size_t)x * V) : 1;
  float a = 0.f;
  if (in && y <= x)
    for (int z = part; z < nsplit; z += LANES) a += partial[(size_t)z * V * V + idx];
  if (LANES == 8) {
    a += __shfl_xor_sync(0xffffffffu, a, 1);
    a += __shfl_xor_sync(0xffffffffu, a, 2);
    a += __shfl_xor_sync(0xffffffffu, a, 4);
  }
  if (!in || y > x || part) return;
  a /= (float)(N - 1);
  Sigma[(size_t)x * V + y] = a;
  Sigma[(size_t)y * V + x] = a;
}

static void launch_syrk_reduce(const float* partial, int nsplit, int V, int N, float* Sigma,
                               const Ctrl* ctrl, int respect_done, cudaStream_t st) {
  ++g_launches;
  const size_t e = (size_t)V * V;
  if (V <= 128)
    launch_pdl(syrk_reduce_kernel<8>, (unsigned)((8 * e + 255) / 256), 256, 0, st, partial, nsplit, V, N,
               Sigma, ctrl, respect_done);
  else
    launch_pdl(syrk_reduce_kernel<1>, (unsigned)((e + 255) / 256), 256, 0, st, partial, nsplit, V, N, Sigma,
               ctrl, respect_done);
}

__global__ void __launch_bounds__(256)
trace_kernel(const float* __restrict__ Sigma, int V, Ctrl* ctrl, int respect_done) {
  __shared__ double scratch[33];
  if (respect_done && ctrl->done) return;
  double a = 0.0;
  for (int x = threadIdx.x; x < V; x += blockDim.x) a += (double)Sigma[(size_t)x * V + x];
  a = block_sum(a, scratch);
  if (threadIdx.x == 0) { ctrl->trace = (float)a; ctrl->chol_fail = 0; }
}

// attempt 0: plain; attempt 1: runs only if attempt 0 failed, adds 1e-6 tr/V to the diagonal.
__device__ __forceinline__ bool chol_skip(const Ctrl* ctrl, int attempt, int respect_done) {
  if (respect_done && ctrl->done) return true;
  return attempt == 1 && !(ctrl->chol_fail & 1);
}

constexpr int CS_NB = 8;               // panel width of the factorisations below

// ---- V <= 160 in one CTA: register-resident state, warp-specialised --------------------------
// Right-looking factorisation in 8-column panels (column block q = columns 8q .. 8q+7), no matrix
// in shared memory.  Two groups of warps:
//  * ROW warps: thread r owns matrix row r.  At panel p it holds x = A[r][8p..8p+7] with every
//    earlier panel applied, re-factorises the 8 x 8 diagonal block in registers with its own row
//    riding along as a ninth row (the pivots are the only serial chain), publishes its eight new
//    L entries k-major (Lp), and then applies panel p to its own entries of the NEXT column block
//    itself: x' = Ap - sum_k x[k] L[8(p+1)+c][k].  The eight rows of the next diagonal block go
//    through shared memory (Dn).  Two row-group barriers per panel; nothing else is on the
//    critical path.
//  * TILE warps: the lower triangle is cut into 4 x 4 tiles, one per thread, in registers for the
//    whole factorisation (<= 820 tiles: 26 warps).  A tile of column block q receives the
//    updates of panels 0 .. q-2 from Lp (sixteen 16-byte shared loads, 128 FMAs per panel) and
//    is then published k-major (Ap) for the row warps, which need it one whole panel later.
//  * one housekeeping warp copies Lp to Lc and writes the zeros above the diagonal.
// Named barriers: AP_FULL (tiles -> rows), LP_FULL (rows -> tiles), LP_EMPTY (tiles -> rows, two
// Lp buffers), ROW_A / ROW_B (row group).  Both attempts of reading A4 run inside this launch.
constexpr int CT_LD = 160;                 // leading dimension of Ap / Lp (rows), V <= 160
constexpr int CT_ROW_WARPS = 5;            // 160 rows
constexpr int CT_TILE_WARPS = 26;          // 40 * 41 / 2 = 820 tiles
constexpr int CT_THREADS = 32 * (CT_TILE_WARPS + CT_ROW_WARPS + 1);   // + 1 housekeeping warp
constexpr int CT_RWT = 32 * CT_ROW_WARPS;
// named barriers: M(p) = "panel p of L is in Lp, column block p + 1 of A is in Ap" (rows, tile
// warps that still hold a tile of a block >= p + 1, housekeeping); B(p) = "the diagonal block of
// panel p + 1 is in Dn, and Lp of panel p - 1 has been read" (rows sync; tile warps and
// housekeeping arrive); AP0 / B_PRO: the same two for the prologue.  M and B alternate ids.
enum { BAR_M = 1, BAR_B = 3, BAR_AP0 = 5, BAR_B_PRO = 6 };

__device__ __forceinline__ void bar_sync(int id, int nthreads) {
  asm volatile("bar.sync %0, %1;" ::"r"(id), "r"(nthreads) : "memory");
}
__device__ __forceinline__ void bar_arrive(int id, int nthreads) {
  asm volatile("bar.arrive %0, %1;" ::"r"(id), "r"(nthreads) : "memory");
}
__device__ __forceinline__ float rsqrt_ftz(float x) {
  float y;
  asm("rsqrt.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x));
  return y;
}

struct CholTiles {
  int nT;                                   // tile rows = ceil(V / 4)
  __device__ int first(int C) const { return C * nT - C * (C - 1) / 2; }   // first tile of column C
  __device__ int ntiles() const { return nT * (nT + 1) / 2; }
  __device__ int nwarps() const { return (ntiles() + 31) >> 5; }
  // tile warps that hold a tile in a column >= C: warps [warp_lo(C), nwarps())
  __device__ int warp_lo(int C) const { return C >= nT ? nwarps() : first(C) >> 5; }
  // number of warps holding a tile of columns C, C + 1 (first of them: warp_lo(C)); 0 if none
  __device__ int owners(int C) const {
    if (C >= nT) return 0;
    const int last = first(min(C + 2, nT)) - 1;
    return (last >> 5) - (first(C) >> 5) + 1;
  }
};

// One factorisation pass of the V x V matrix S (row stride s_ld, lower triangle read) by a CTA of
// CT_THREADS threads; L goes to `out` (row stride o_ld: global or shared memory), with zeros above
// the diagonal if zero_upper.  *failed_s is set if a pivot fails.  Ends without a block barrier.
__device__ __forceinline__ void chol_tiles_pass(const float* __restrict__ S, int s_ld, float* out, int o_ld,
                                                int V, float add, bool zero_upper,
                                                float (*Ap)[CS_NB * CT_LD], float (*Lp)[CS_NB * CT_LD],
                                                float (*Dn)[CS_NB * CS_NB], int* failed_s) {
  const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
  CholTiles T;
  T.nT = (V + 3) >> 2;
  const int ntiles = T.ntiles(), ntw = T.nwarps();
  const int nP = (V + CS_NB - 1) / CS_NB;
  const bool is_tile = warp < CT_TILE_WARPS, is_row = !is_tile && warp < CT_TILE_WARPS + CT_ROW_WARPS;
  // tile of this thread (numbered column by column: t -> column C ascending, rows R >= C)
  int R = 0, C = 0;
  const bool has_tile = is_tile && tid < ntiles;
  if (has_tile) {
    int ur, uc;
    tri_tile(ntiles - 1 - tid, ur, uc);      // row-major lower index of the mirrored tile
    C = T.nT - 1 - ur;
    R = T.nT - 1 - uc;
  }
  const int r0 = 4 * R, c0 = 4 * C, q = C >> 1;
  if (is_tile) {
    if (warp >= ntw && zero_upper)        // idle tile warps: zeros above the diagonal
      for (int x = warp - ntw; x < V; x += CT_TILE_WARPS - ntw)
        for (int y = x + 1 + lane; y < V; y += 32) out[(size_t)x * o_ld + y] = 0.f;
    if (warp < ntw) {
      float a[4][4];
#pragma unroll
      for (int i = 0; i < 4; ++i)
#pragma unroll
        for (int j = 0; j < 4; ++j) {
          const int x = r0 + i, y = c0 + j;
          const float v = S[(size_t)min(x, V - 1) * s_ld + min(y, V - 1)];   // always in range
          a[i][j] = (x < V && y < V) ? v + (x == y ? add : 0.f) : (x == y ? 1.f : 0.f);
        }
      // column blocks 0 and 1 receive no update from a tile warp: publish them right away
      if (has_tile && q <= 1) {
        float* dst = &Ap[q][(c0 - 8 * q) * CT_LD + r0];
#pragma unroll
        for (int j = 0; j < 4; ++j)
          *reinterpret_cast<float4*>(dst + j * CT_LD) = make_float4(a[0][j], a[1][j], a[2][j], a[3][j]);
      }
      if (warp < T.owners(0)) bar_arrive(BAR_AP0, 32 * T.owners(0) + CT_RWT);
      for (int p = 0; p < nP; ++p) {
        const int lo1 = T.warp_lo(2 * p + 2), alo = T.warp_lo(2 * p + 4), buf = p & 1;
        const int nM = 32 * (ntw - lo1) + 32 + CT_RWT;
        if (warp < alo) {                                   // every tile of this warp is final
          if (warp >= lo1) bar_arrive(BAR_M + buf, nM);     // (its block p + 1 tiles are in Ap)
          break;
        }
        bar_sync(BAR_M + buf, nM);
        // update from panel p for the tiles of column blocks >= p + 2
        if (has_tile && q >= p + 2) {
          const float* lp = &Lp[buf][0];
#pragma unroll
          for (int k = 0; k < CS_NB; ++k) {
            const float4 lr = *reinterpret_cast<const float4*>(lp + k * CT_LD + r0);
            const float4 lc = *reinterpret_cast<const float4*>(lp + k * CT_LD + c0);
            const float lrv[4] = {lr.x, lr.y, lr.z, lr.w}, lcv[4] = {lc.x, lc.y, lc.z, lc.w};
#pragma unroll
            for (int i = 0; i < 4; ++i)
#pragma unroll
              for (int j = 0; j < 4; ++j) a[i][j] = fmaf(-lrv[i], lcv[j], a[i][j]);
          }
        }
        bar_arrive(BAR_B + (buf ^ 1), 32 * (ntw - alo) + 32 + CT_RWT);   // B(p + 1): Lp[buf] read
        // column block p + 2 is complete now: publish it (visible through M(p + 1))
        if (has_tile && q == p + 2) {
          float* dst = &Ap[q & 1][(c0 - 8 * q) * CT_LD + r0];
#pragma unroll
          for (int j = 0; j < 4; ++j)
            *reinterpret_cast<float4*>(dst + j * CT_LD) = make_float4(a[0][j], a[1][j], a[2][j], a[3][j]);
        }
      }
    }
  } else if (is_row) {
    const int r = tid - 32 * CT_TILE_WARPS;          // matrix row of this thread (fixed)
    const bool live = r < CS_NB * nP;                // rows of the matrix padded to whole panels
    if (r == 0) *failed_s = 0;
    // rows [V, 4 nT) exist in the tiles as identity padding: their L entries are zero
    if (r >= V) {
#pragma unroll
      for (int k = 0; k < 2 * CS_NB; ++k) (&Lp[0][0])[k * CT_LD + r] = 0.f;
    }
    float x[CS_NB];
    bar_sync(BAR_AP0, 32 * T.owners(0) + CT_RWT);
#pragma unroll
    for (int k = 0; k < CS_NB; ++k) x[k] = (r < V) ? Ap[0][k * CT_LD + r] : (k == r ? 1.f : 0.f);
    if (r < CS_NB) {
#pragma unroll
      for (int k = 0; k < CS_NB; ++k) Dn[0][k * CS_NB + r] = x[k];
    }
    bar_sync(BAR_B_PRO, CT_RWT);
    for (int p = 0; p < nP; ++p) {
      const int buf = p & 1, jb = CS_NB * p, ri = r - jb;
      if (ri >= 0 && live) {
        const float* dn = &Dn[buf][0];
        float D[CS_NB][CS_NB];
#pragma unroll
        for (int k = 0; k < CS_NB; ++k) {
          const float4 lo = *reinterpret_cast<const float4*>(dn + k * CS_NB);
          const float4 hi = *reinterpret_cast<const float4*>(dn + k * CS_NB + 4);
          D[0][k] = lo.x; D[1][k] = lo.y; D[2][k] = lo.z; D[3][k] = lo.w;
          D[4][k] = hi.x; D[5][k] = hi.y; D[6][k] = hi.z; D[7][k] = hi.w;
        }
        bool bad = false;
#pragma unroll
        for (int k = 0; k < CS_NB; ++k) {
          // pivots below the smallest normal number count as failures (the reciprocal square
          // root flushes them); 1/sqrt(d) = SFU seed + one Newton step (~1 ulp)
          const float d0 = D[k][k];
          const bool ok = d0 >= 1.17549435e-38f;
          bad |= !ok;
          const float d = ok ? d0 : 1.f;
          float inv = rsqrt_ftz(d0);
          inv = ok ? inv : 1.f;
          inv = inv * fmaf(-0.5f * d * inv, inv, 1.5f);
          D[k][k] = d * inv;
#pragma unroll
          for (int i = k + 1; i < CS_NB; ++i) D[i][k] *= inv;
          x[k] *= inv;
#pragma unroll
          for (int i = k + 1; i < CS_NB; ++i)
#pragma unroll
            for (int c = k + 1; c <= i; ++c) D[i][c] = fmaf(-D[i][k], D[c][k], D[i][c]);
#pragma unroll
          for (int c = k + 1; c < CS_NB; ++c) x[c] = fmaf(-x[k], D[c][k], x[c]);
        }
        if (bad) *failed_s = 1;
        // rows of the diagonal block: their elimination reproduces the factor; zero above it
#pragma unroll
        for (int k = 1; k < CS_NB; ++k) if (k > ri) x[k] = 0.f;
        float* lp = &Lp[buf][0];
#pragma unroll
        for (int k = 0; k < CS_NB; ++k) lp[k * CT_LD + r] = x[k];
      }
      const int nM = 32 * (ntw - T.warp_lo(2 * p + 2)) + 32 + CT_RWT;
      if (p + 1 == nP) { bar_arrive(BAR_M + buf, nM); break; }
      bar_sync(BAR_M + buf, nM);
      if (ri >= CS_NB && live) {
        // own entries of column block p + 1: A (panels < p applied by the tiles) minus panel p
        const float* lp = &Lp[buf][jb + CS_NB];
        const float* ap = &Ap[buf ^ 1][0];
        float xn[CS_NB];
#pragma unroll
        for (int c = 0; c < CS_NB; ++c)
          xn[c] = (r < V) ? ap[c * CT_LD + r] : (c == ri - CS_NB ? 1.f : 0.f);
#pragma unroll
        for (int k = 0; k < CS_NB; ++k) {
          const float4 lo = *reinterpret_cast<const float4*>(lp + k * CT_LD);
          const float4 hi = *reinterpret_cast<const float4*>(lp + k * CT_LD + 4);
          const float l[CS_NB] = {lo.x, lo.y, lo.z, lo.w, hi.x, hi.y, hi.z, hi.w};
#pragma unroll
          for (int c = 0; c < CS_NB; ++c) xn[c] = fmaf(-x[k], l[c], xn[c]);
        }
#pragma unroll
        for (int c = 0; c < CS_NB; ++c) x[c] = xn[c];
        if (ri < 2 * CS_NB) {
#pragma unroll
          for (int c = 0; c < CS_NB; ++c) Dn[buf ^ 1][c * CS_NB + ri - CS_NB] = x[c];
        }
      }
      // B(p): next diagonal block visible; readers of Lp[buf ^ 1] (panel p - 1) are done
      bar_sync(BAR_B + buf, CT_RWT + (p >= 1 ? 32 * (ntw - T.warp_lo(2 * p + 2)) + 32 : 0));
    }
  } else {
    // housekeeping warp: L from Lp to Lc panel by panel (and the zeros above the diagonal if
    // every tile warp holds tiles)
    if (zero_upper && ntw == CT_TILE_WARPS)
      for (int x = 0; x < V; ++x)
        for (int y = x + 1 + lane; y < V; y += 32) out[(size_t)x * o_ld + y] = 0.f;
    for (int p = 0; p < nP; ++p) {
      const int buf = p & 1, jb = CS_NB * p;
      bar_sync(BAR_M + buf, 32 * (ntw - T.warp_lo(2 * p + 2)) + 32 + CT_RWT);
      const float* lp = &Lp[buf][0];
      for (int r = jb + lane; r < V; r += 32) {
#pragma unroll
        for (int k = 0; k < CS_NB; ++k)
          if (jb + k < V && jb + k <= r) out[(size_t)r * o_ld + jb + k] = lp[k * CT_LD + r];
      }
      if (p + 2 < nP) bar_arrive(BAR_B + (buf ^ 1), 32 * (ntw - T.warp_lo(2 * p + 4)) + 32 + CT_RWT);
    }
  }
}

__global__ void __launch_bounds__(CT_THREADS)
chol_small_kernel(const float* __restrict__ Sigma, float* __restrict__ Lc, int V, Ctrl* ctrl,
                  int respect_done) {
  pdl_enter();
  __shared__ __align__(16) float Ap[2][CS_NB * CT_LD];   // column block q of A, k-major, buffer q & 1
  __shared__ __align__(16) float Lp[2][CS_NB * CT_LD];   // panel p of L, k-major, buffer p & 1
  __shared__ __align__(16) float Dn[2][CS_NB * CS_NB];   // diagonal block of panel p, k-major
  __shared__ int failed_s;
  if (respect_done && ctrl->done) return;
  const int tid = threadIdx.x, lane = tid & 31;
  float tr = 0.f;
  int status = 0;
  for (int attempt = 0; attempt < 2; ++attempt) {
    if (attempt) {                            // jitter scale of reading A4 (only if attempt 0 failed)
      double t2 = 0.0;
      for (int x = lane; x < V; x += 32) t2 += (double)Sigma[(size_t)x * V + x];
#pragma unroll
      for (int o = 16; o > 0; o >>= 1) t2 += __shfl_xor_sync(0xffffffffu, t2, o);
      tr = (float)t2;
    }
    const float add = attempt ? 1e-6f * tr / (float)V : 0.f;
    chol_tiles_pass(Sigma, V, Lc, V, V, add, attempt == 0, Ap, Lp, Dn, &failed_s);
    __syncthreads();
    const int failed = failed_s;
    __syncthreads();
    if (!failed) { status = attempt; break; }
    status = -1;
  }
  if (tid == 0) {
    ctrl->chol_status = status; ctrl->chol_fail = 0;
    if (status != 0) ctrl->trace = tr;
  }
}

// ------------------------------------------------------------------ large V: blocked ---------
__global__ void chol_copy_kernel(const float* __restrict__ Sigma, float* __restrict__ Lc, int V,
                                 const Ctrl* ctrl, int attempt, int respect_done) {
  if (chol_skip(ctrl, attempt, respect_done)) return;
  int idx = blockIdx.x * blockDim.x + threadIdx.x;
  if (idx >= V * V) return;
  int x = idx / V, y = idx - x * V;
  float add = (attempt && x == y) ? 1e-6f * ctrl->trace / (float)V : 0.f;
  Lc[idx] = (y <= x) ? Sigma[idx] + add : 0.f;
}

// Diagonal block [j0, j0+nb) factorised in place by one CTA (register tiles, chol_tiles_pass: every
// entry is in registers before the first result is stored).
__global__ void __launch_bounds__(CT_THREADS)
chol_diag_kernel(float* __restrict__ A, int V, int j0, Ctrl* ctrl, int attempt,
                 int respect_done) {
  __shared__ __align__(16) float Ap[2][CS_NB * CT_LD];
  __shared__ __align__(16) float Lp[2][CS_NB * CT_LD];
  __shared__ __align__(16) float Dn[2][CS_NB * CS_NB];
  __shared__ int failed_s;
  if (chol_skip(ctrl, attempt, respect_done)) return;
  const int nb = min(64, V - j0);
  float* blk = A + (size_t)j0 * V + j0;
  chol_tiles_pass(blk, V, blk, V, nb, 0.f, false, Ap, Lp, Dn, &failed_s);
  __syncthreads();
  if (threadIdx.x == 0 && failed_s) atomicOr(&ctrl->chol_fail, attempt ? 2 : 1);
}

// Rows below the diagonal block: X L11^T = A21, one thread per row.  Right-looking: once x_c is
// known (one multiplication by the tabulated 1 / l_cc) the 63 - c updates x_m -= x_c l_mc are
// independent; L11 sits transposed in shared memory (Tt[c][m] = l_mc: 16-byte broadcast loads).
__global__ void __launch_bounds__(64)
chol_trsm_kernel(float* __restrict__ A, int V, int j0, const Ctrl* ctrl, int attempt,
                 int respect_done) {
  __shared__ __align__(16) float Tt[64][64];
  __shared__ float inv[64];
  if (chol_skip(ctrl, attempt, respect_done)) return;
  const int nb = min(64, V - j0), t = threadIdx.x;
  for (int c = 0; c < 64; ++c)                       // thread t: row t of L11 -> column t of Tt
    Tt[c][t] = (t < nb && c <= t) ? A[(size_t)(j0 + t) * V + j0 + c] : 0.f;
  inv[t] = t < nb ? 1.0f / A[(size_t)(j0 + t) * V + j0 + t] : 0.f;
  __syncthreads();
  const int row = j0 + nb + blockIdx.x * 64 + t;
  if (row >= V) return;
  float x[64];
  float* a = A + (size_t)row * V + j0;
  if (nb == 64 && (V & 3) == 0) {
#pragma unroll
    for (int c = 0; c < 64; c += 4) {
      const float4 v = *reinterpret_cast<const float4*>(a + c);
      x[c] = v.x; x[c + 1] = v.y; x[c + 2] = v.z; x[c + 3] = v.w;
    }
  } else {
#pragma unroll
    for (int c = 0; c < 64; ++c) x[c] = c < nb ? a[c] : 0.f;
  }
#pragma unroll
  for (int c = 0; c < 64; ++c) {
    x[c] *= inv[c];                                  // (columns >= nb: inv = 0, x = 0)
#pragma unroll
    for (int m4 = (c + 1) & ~3; m4 < 64; m4 += 4) {
      const float4 l = *reinterpret_cast<const float4*>(&Tt[c][m4]);
      if (m4 > c) x[m4] = fmaf(-x[c], l.x, x[m4]);
      if (m4 + 1 > c) x[m4 + 1] = fmaf(-x[c], l.y, x[m4 + 1]);
      if (m4 + 2 > c) x[m4 + 2] = fmaf(-x[c], l.z, x[m4 + 2]);
      x[m4 + 3] = fmaf(-x[c], l.w, x[m4 + 3]);
    }
  }
  if (nb == 64 && (V & 3) == 0) {
#pragma unroll
    for (int c = 0; c < 64; c += 4) *reinterpret_cast<float4*>(a + c) = make_float4(x[c], x[c + 1], x[c + 2], x[c + 3]);
  } else {
#pragma unroll
    for (int c = 0; c < 64; ++c)
      if (c < nb) a[c] = x[c];
  }
}

// Trailing update A22 -= L21 L21^T on the lower-triangular 64x64 tiles of rows/cols >= j1.
__global__ void __launch_bounds__(256)
chol_update_kernel(float* __restrict__ A, int V, int j0, int j1, const Ctrl* ctrl, int attempt,
                   int respect_done) {
  if (chol_skip(ctrl, attempt, respect_done)) return;
  __shared__ __align__(16) float As[16][68], Bs[16][68];
  int tr, tc;
  tri_tile(blockIdx.x, tr, tc);
  const int x0 = j1 + tr * 64, y0 = j1 + tc * 64;
  float acc[4][4];
#pragma unroll
  for (int p = 0; p < 4; ++p)
#pragma unroll
    for (int r = 0; r < 4; ++r) acc[p][r] = 0.f;
  nt_tile<false>(A, (size_t)V, x0, y0, V, j0, j1, V, nullptr, acc, As, Bs);
  const int tx = threadIdx.x & 15, ty = threadIdx.x >> 4;
#pragma unroll
  for (int p = 0; p < 4; ++p)
#pragma unroll
    for (int r = 0; r < 4; ++r) {
      int x = x0 + ty * 4 + p, y = y0 + tx * 4 + r;
      if (x < V && y <= x) A[(size_t)x * V + y] -= acc[p][r];
    }
}

__global__ void chol_finalize_kernel(Ctrl* ctrl, int respect_done) {
  if (respect_done && ctrl->done) return;
  int f = ctrl->chol_fail;
  ctrl->chol_status = (f == 0) ? 0 : ((f & 2) ? -1 : 1);
  ctrl->chol_fail = 0;
}

void launch_cholesky(const float* Sigma, float* Lc, int V, Ctrl* ctrl, int respect_done,
                     cudaStream_t st) {
  if (V <= CT_LD) {
    ++g_launches; launch_pdl(chol_small_kernel, 1, CT_THREADS, 0, st, Sigma, Lc, V, ctrl, respect_done);
    return;
  }
  ++g_launches; trace_kernel<<<1, 256, 0, st>>>(Sigma, V, ctrl, respect_done);
  for (int attempt = 0; attempt < 2; ++attempt) {
    ++g_launches; chol_copy_kernel<<<(V * V + 255) / 256, 256, 0, st>>>(Sigma, Lc, V, ctrl, attempt,
                                                          respect_done);
    for (int j0 = 0; j0 < V; j0 += 64) {
      int j1 = min(V, j0 + 64);
      ++g_launches; chol_diag_kernel<<<1, CT_THREADS, 0, st>>>(Lc, V, j0, ctrl, attempt, respect_done);
      int rows = V - j1;
      if (rows > 0) {
        ++g_launches; chol_trsm_kernel<<<(rows + 63) / 64, 64, 0, st>>>(Lc, V, j0, ctrl, attempt,
                                                          respect_done);
        int nt = (rows + 63) / 64;
        ++g_launches; chol_update_kernel<<<nt * (nt + 1) / 2, 256, 0, st>>>(Lc, V, j0, j1, ctrl, attempt,
                                                              respect_done);
      }
    }
  }
  ++g_launches; chol_finalize_kernel<<<1, 1, 0, st>>>(ctrl, respect_done);
}

static int cov_nsplit(int V, int N) {
  int nt = (V + 63) / 64;
  int tiles = nt * (nt + 1) / 2;
  int want = (2 * 148 + tiles - 1) / tiles;
  int maxsplit = (round_up(N, 128) + 127) / 128;   // chunks of >= 128 particles
  int ns = want < 1 ? 1 : want;
  if (ns > maxsplit) ns = maxsplit;
  if (ns > 128) ns = 128;
  return ns;
}

size_t cov_partial_floats(int V, int N) {
  int ns = cov_nsplit(V, N);
  const int ld = round_up(N, 128);
  if (syrk_tc_supported(V, ld) && syrk_tc_nsplit(V, ld, false) > ns) ns = syrk_tc_nsplit(V, ld, false);
  if (syrk_tc_supported(V, ld) && syrk_tc_nsplit(V, ld, true) > ns) ns = syrk_tc_nsplit(V, ld, true);
  if (syrk_tc_small_supported(V, ld) && syrk_tc_small_nsplit(ld) > ns) ns = syrk_tc_small_nsplit(ld);
  return (size_t)ns * V * V;
}

void launch_cov_chol(const CovCholArgs& a, cudaStream_t st) {
  const int V = a.V;
  if (a.tc_scratch && syrk_tc_supported(V, a.ld)) {
    ++g_launches;
    if (a.tc_f16)
      launch_pdl(mean_kernel<true>, V, 256, 0, st, a.phi, a.N, a.ld, a.mu, syrk_tc_amax(a.tc_scratch, V, a.ld),
                 (const Ctrl*)a.ctrl, a.respect_done);
    else
      launch_pdl(mean_kernel<false>, V, 256, 0, st, a.phi, a.N, a.ld, a.mu, (float*)nullptr, (const Ctrl*)a.ctrl,
                 a.respect_done);
    launch_syrk_tc(a.phi, a.N, a.ld, V, a.mu, a.tc_scratch, a.partial, a.ctrl, a.respect_done, st, a.tc_f16);
    launch_syrk_reduce(a.partial, syrk_tc_nsplit(V, a.ld, a.tc_f16), V, a.N, a.Sigma, a.ctrl, a.respect_done, st);
    launch_cholesky(a.Sigma, a.Lc, V, a.ctrl, a.respect_done, st);
    return;
  }
  ++g_launches; launch_pdl(mean_kernel<false>, V, 256, 0, st, a.phi, a.N, a.ld, a.mu, (float*)nullptr,
                           (const Ctrl*)a.ctrl, a.respect_done);
  // (populations below 8192 stay on the SIMT tiles: at n_live = 4096 the 32 tensor-core CTAs take
  // 11 us against 10 for the 3 x 94 SIMT blocks; at N = 16384 it is 11 against 19)
  if (a.tc_small && a.ld >= 8192 && syrk_tc_small_supported(V, a.ld)) {
    launch_syrk_tc_small(a.phi, a.N, a.ld, V, a.mu, a.partial, a.ctrl, a.respect_done, st);
    launch_syrk_reduce(a.partial, syrk_tc_small_nsplit(a.ld), V, a.N, a.Sigma, a.ctrl, a.respect_done, st);
    launch_cholesky(a.Sigma, a.Lc, V, a.ctrl, a.respect_done, st);
    return;
  }
  int ns = cov_nsplit(V, a.N);
  int chunk = round_up((a.ld + ns - 1) / ns, 16);
  ns = (a.ld + chunk - 1) / chunk;
  int nt = (V + 63) / 64;
  dim3 grid(nt * (nt + 1) / 2, ns);
  ++g_launches; launch_pdl(syrk_partial_kernel, grid, 256, 0, st, a.phi, a.N, a.ld, V, a.mu, a.partial, chunk, a.ctrl,
                                            a.respect_done);
  launch_syrk_reduce(a.partial, ns, V, a.N, a.Sigma, a.ctrl, a.respect_done, st);
  launch_cholesky(a.Sigma, a.Lc, V, a.ctrl, a.respect_done, st);
}

}  // namespace phi4
