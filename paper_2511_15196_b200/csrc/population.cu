// population.cu -- the population step P1-P4: next beta by ESS bisection,
// incremental weights + log Z, exact integer systematic resampling, gather.
#include "kernels.cuh"
#include "philox.cuh"

namespace phi4 {

// ---------------------------------------------------------------------------------------------
// P1 + P2 in one CTA (N <= a few 1e5 floats: the vector is L2/L1 resident, and for N <= 16384 it
// is held in registers across all passes).
// R3: f(d) = ESS(d)/N - target, ESS(d) = (sum e^{-d S})^2 / sum e^{-2 d S}; if f(1-beta) >= 0 the
// step is final (beta' = 1), else delta is the root of f on (0, 1-beta) -- R3 defines it as the
// limit of 48 bisection halvings.  f is smooth and strictly decreasing, so a bracketed Newton
// iteration on h(d) = log ESS(d)/N - log target (close to a parabola in d: ESS/N = exp(-d^2 var S)
// for Gaussian S) started from the previous temperature's delta reaches the same root to 1e-7
// relative in 3-5 evaluations; each evaluation is one pass over the N actions that also yields
// h'(d) = 2 a'/a - b'/b from a' = -sum x e, b' = -2 sum x e^2 (x = S - S_min, e = e^{-d x}).
// A step that leaves the bracket falls back to bisection (reading R3).
// Then w_i = exp(-d (S_i - S_min)) (max w = 1) and
// dlogZ = -d S_min + log sum w - log N   (U0 cancels between p_beta and p_beta').
// ---------------------------------------------------------------------------------------------
// floor(w 2^40) for an fp32 w in [0, 1], from the bits: w = m 2^(e-150), so q = m 2^(e-110).
// Exact (reading R5: identical to floor((double)w * 2^40)).
__device__ __forceinline__ unsigned long long quantise40(float w) {
  const uint32_t b = __float_as_uint(w);
  const int e = (int)((b >> 23) & 0xffu);
  if (e == 0 || (b >> 31)) return 0ull;                       // zero, subnormal (< 2^-126) or negative
  const unsigned long long m = (unsigned long long)((b & 0x7fffffu) | 0x800000u);
  const int sh = e - 110;
  return sh >= 0 ? (m << sh) : (sh > -24 ? (m >> (-sh)) : 0ull);
}

namespace rw {
constexpr int THREADS = 1024, RC = 16;        // register cache: up to 16 actions per thread
}

struct EssSums { double a, b, da, db; };

// all four sums for one d: e_i by ex2.approx on the max-shifted argument (relative error ~1e-6 |x|
// on weights that matter, far below the 1e-4 tolerance of the root), per-thread partials in FP32
// (<= 16 terms when cached, folded every 32 terms otherwise), block reduction in FP64
template <bool CACHED>
__device__ __forceinline__ EssSums ess_sums(const float (&xs)[rw::RC], int cnt,
                                            const float* __restrict__ S, int N, float smin,
                                            double d, double4* scratch) {
  const float df = (float)d * 1.4426950408889634f;
  double A = 0.0, B = 0.0, DA = 0.0, DB = 0.0;
  if (CACHED) {
    float a = 0.f, b = 0.f, da = 0.f, db = 0.f;
#pragma unroll
    for (int j = 0; j < rw::RC; ++j)
      if (j < cnt) {
        float e;
        asm("ex2.approx.ftz.f32 %0, %1;" : "=f"(e) : "f"(-df * xs[j]));
        const float e2 = e * e;
        a += e; b += e2;
        da = fmaf(xs[j], e, da); db = fmaf(xs[j], e2, db);
      }
    A = a; B = b; DA = da; DB = db;
  } else {
    for (int i0 = threadIdx.x; i0 < N; i0 += rw::THREADS * 32) {
      float a = 0.f, b = 0.f, da = 0.f, db = 0.f;
      for (int j = 0; j < 32; ++j) {
        const int i = i0 + j * rw::THREADS;
        if (i < N) {
          const float x = S[i] - smin;
          float e;
          asm("ex2.approx.ftz.f32 %0, %1;" : "=f"(e) : "f"(-df * x));
          const float e2 = e * e;
          a += e; b += e2;
          da = fmaf(x, e, da); db = fmaf(x, e2, db);
        }
      }
      A += a; B += b; DA += da; DB += db;
    }
  }
  const int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
  A = warp_sum(A); B = warp_sum(B); DA = warp_sum(DA); DB = warp_sum(DB);
  if (lane == 0) scratch[w] = make_double4(A, B, DA, DB);
  __syncthreads();
  EssSums r{0.0, 0.0, 0.0, 0.0};
  if (w == 0) {                                    // the totals are valid in warp 0 only
    double4 t = scratch[lane];                     // 1024 threads: exactly 32 warps
    r.a = warp_sum(t.x); r.b = warp_sum(t.y); r.da = -warp_sum(t.z); r.db = -2.0 * warp_sum(t.w);
  }
  return r;
}

template <bool CACHED>
__device__ __forceinline__ void next_delta_reweight_body(const float* __restrict__ S, int N,
                                                         float ess_target, double delta_fixed,
                                                         float* __restrict__ w,
                                                         unsigned long long* __restrict__ C,
                                                         Ctrl* ctrl) {
  __shared__ double4 scratch[33];
  __shared__ float smin_s[33];
  __shared__ double bcast_x;
  __shared__ int bcast_flags;
  float xs[rw::RC];
  int cnt = 0;
  float m = INFINITY;
  // cached layout: warp w owns the contiguous span [w 32 ipt, (w+1) 32 ipt), lane l its elements
  // l, l + 32, ...: every load / store instruction covers 32 consecutive entries, and the integer
  // scan of P3 is a warp scan per row plus a running carry
  const int ipt = min(rw::RC, (N + rw::THREADS - 1) / rw::THREADS);
  const int run0 = (int)(threadIdx.x >> 5) * 32 * ipt + (int)(threadIdx.x & 31);
  if (CACHED) {
    cnt = max(0, min(ipt, (N - run0 + 31) >> 5));
#pragma unroll
    for (int j = 0; j < rw::RC; ++j) {
      xs[j] = j < cnt ? S[run0 + 32 * j] : INFINITY;
      m = fminf(m, xs[j]);
    }
  } else {
    for (int i = threadIdx.x; i < N; i += rw::THREADS) m = fminf(m, S[i]);
  }
  m = warp_min(m);
  if ((threadIdx.x & 31) == 0) smin_s[threadIdx.x >> 5] = m;
  __syncthreads();
  if (threadIdx.x < 32) {
    float v = warp_min(smin_s[threadIdx.x]);
    if (threadIdx.x == 0) smin_s[32] = v;
  }
  __syncthreads();
  const float smin = smin_s[32];
  if (CACHED) {
#pragma unroll
    for (int j = 0; j < rw::RC; ++j) xs[j] -= smin;
  }
  const double beta = ctrl->beta;
  const double rest = 1.0 - beta;
  const double ltarget = log((double)ess_target), lN = log((double)N);
  double delta;
  int final_step = 0;
  if (delta_fixed >= 0.0) {
    delta = delta_fixed;
    final_step = (beta + delta >= 1.0);
  } else {
    // thread 0 owns the bracket and the Newton step (FP64 logs and divisions once, not 1024
    // times); the next abscissa and the stop flag go through shared memory
    double lo = 0.0, hi = rest;
    bool hi_known = false;                           // sign of h(rest) not evaluated yet
    const double prev = ctrl->delta;
    double x = (prev > 0.0 && prev < rest) ? prev : rest;
    delta = rest;
    for (int it = 0; it < 64; ++it) {
      const EssSums q = ess_sums<CACHED>(xs, cnt, S, N, smin, x, scratch);
      if (threadIdx.x == 0) {
        int stop = 0, fin = 0;
        double xn = x;
        const double h = 2.0 * log(q.a) - log(q.b) - lN - ltarget;
        if (x >= rest && !hi_known) {
          if (h >= 0.0) { stop = 1; fin = 1; xn = rest; }
          hi_known = true;
        }
        if (!stop) {
          if (h > 0.0) lo = x; else hi = x;
          if (fabs(h) < 1e-9) stop = 1;
          else {
            const double dh = 2.0 * q.da / q.a - q.db / q.b;
            xn = x - h / dh;
            if (!(xn > lo && xn < hi)) {
              if (!hi_known && xn >= hi) xn = rest;      // probe the end of the interval
              else if (hi_known) xn = 0.5 * (lo + hi);
              else xn = fmin(rest, 2.0 * x);             // dh >= 0 or NaN far out: walk right
            }
            if (fabs(xn - x) <= 1e-7 * xn && !(xn >= rest && !hi_known)) stop = 1;
          }
        }
        bcast_x = xn; bcast_flags = stop | (fin << 1);
      }
      __syncthreads();
      x = bcast_x;
      delta = x;
      const int fl = bcast_flags;
      final_step = fl >> 1;
      if (fl & 1) break;
    }
  }
  const float df = (float)delta;
  double a = 0.0, b = 0.0;
  if (CACHED) {
    unsigned long long run = 0;
#pragma unroll
    for (int j = 0; j < rw::RC; ++j)
      if (j < cnt) {
        const float e = expf(-df * xs[j]);
        xs[j] = e;                                   // kept for the scan below
        w[run0 + 32 * j] = e;
        a += (double)e;
        b += (double)e * (double)e;
        run += quantise40(e);
      }
    if (C) {
      // P3 fused (reading R5): inclusive integer scan of q_i = floor(w_i 2^40).  Warp totals ->
      // exclusive offsets of the warp spans; inside a span, one warp scan per row of 32.
      __shared__ unsigned long long wsum[32];
      const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
      unsigned long long tot = run;
#pragma unroll
      for (int o = 16; o > 0; o >>= 1) tot += __shfl_xor_sync(0xffffffffu, tot, o);
      if (lane == 0) wsum[wid] = tot;
      __syncthreads();
      if (wid == 0) {
        unsigned long long v = wsum[lane], sc = v;
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) {
          unsigned long long u = __shfl_up_sync(0xffffffffu, sc, o);
          if (lane >= o) sc += u;
        }
        wsum[lane] = sc - v;  // exclusive
      }
      __syncthreads();
      unsigned long long carry = wsum[wid];
#pragma unroll
      for (int j = 0; j < rw::RC; ++j)
        if (j < ipt) {                               // block-uniform bound: shuffles stay convergent
          unsigned long long inc = j < cnt ? quantise40(xs[j]) : 0ull;
#pragma unroll
          for (int o = 1; o < 32; o <<= 1) {
            unsigned long long v = __shfl_up_sync(0xffffffffu, inc, o);
            if (lane >= o) inc += v;
          }
          if (j < cnt) C[run0 + 32 * j] = carry + inc;
          carry += __shfl_sync(0xffffffffu, inc, 31);
        }
      if (threadIdx.x == rw::THREADS - 1) {
        ctrl->q_total = carry;
        if (carry == 0ull) ctrl->nan_flag = 1;
      }
    }
  } else {
    for (int i = threadIdx.x; i < N; i += rw::THREADS) {
      const float e = expf(-df * (S[i] - smin));
      w[i] = e;
      a += (double)e;
      b += (double)e * (double)e;
    }
  }
  {
    const int lane = threadIdx.x & 31, wi = threadIdx.x >> 5;
    a = warp_sum(a);
    b = warp_sum(b);
    __syncthreads();
    if (lane == 0) scratch[wi] = make_double4(a, b, 0.0, 0.0);
    __syncthreads();
    if (wi == 0) {
      double4 t = scratch[lane];
      t.x = warp_sum(t.x);
      t.y = warp_sum(t.y);
      if (lane == 0) scratch[32] = t;
    }
    __syncthreads();
    a = scratch[32].x;
    b = scratch[32].y;
  }
  if (threadIdx.x == 0) {
    double dlz = -delta * (double)smin + log(a) - lN;
    ctrl->delta = delta;
    ctrl->beta = final_step ? 1.0 : beta + delta;
    ctrl->ess_frac = a * a / (b * (double)N);
    ctrl->dlogZ = dlz;
    ctrl->logZ += dlz;
    ctrl->S_min = smin;
    if (!isfinite(dlz)) ctrl->nan_flag = 1;
  }
}

__global__ void __launch_bounds__(rw::THREADS)
next_delta_reweight_kernel(const float* __restrict__ S, int N, float ess_target,
                           double delta_fixed, float* __restrict__ w,
                           unsigned long long* __restrict__ C, Ctrl* ctrl) {
  pdl_enter();
  if (ctrl->done) return;
  if (N <= rw::THREADS * rw::RC) next_delta_reweight_body<true>(S, N, ess_target, delta_fixed, w, C, ctrl);
  else next_delta_reweight_body<false>(S, N, ess_target, delta_fixed, w, nullptr, ctrl);
}

// C != nullptr and N <= 16384: the integer scan of P3 runs in the same kernel (the weights are
// still in registers); returns whether it did, so that the caller can skip launch_quantise_scan.
bool launch_next_delta_reweight(const float* S, int N, float ess_target, double delta_fixed,
                                float* w, unsigned long long* C, Ctrl* ctrl, cudaStream_t st) {
  const bool fused = C != nullptr && N <= rw::THREADS * rw::RC;
  ++g_launches;
  launch_pdl(next_delta_reweight_kernel, 1, rw::THREADS, 0, st, S, N, ess_target, delta_fixed, w,
             fused ? C : (unsigned long long*)nullptr, ctrl);
  return fused;
}

// ---------------------------------------------------------------------------------------------
// P3, reading R5: q_i = floor(w_i 2^40) (exact: a power-of-two scaling of an fp32), inclusive
// integer scan C_i, T = C_{N-1}.  Integer addition is associative, so the result is the same
// for every scan shape: one CTA, each thread a contiguous run, warp-shuffle scan of the run sums.
// ---------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(1024)
quantise_scan_kernel(const float* __restrict__ w, int N, unsigned long long* __restrict__ C,
                     Ctrl* ctrl) {
  pdl_enter();
  __shared__ unsigned long long wsum[32];
  if (ctrl->done) return;
  const int ipt = (N + blockDim.x - 1) / blockDim.x;
  const int lo = min(N, (int)threadIdx.x * ipt), hi = min(N, lo + ipt);
  unsigned long long run = 0;
  const bool vec = (ipt & 3) == 0 && hi - lo == ipt;     // whole, 16-byte aligned runs
  if (vec) {
    const float4* w4 = reinterpret_cast<const float4*>(w + lo);
    for (int i = 0; i < ipt / 4; ++i) {
      float4 v = w4[i];
      run += quantise40(v.x) +
             quantise40(v.y) +
             quantise40(v.z) +
             quantise40(v.w);
    }
  } else {
    for (int i = lo; i < hi; ++i) run += quantise40(w[i]);
  }
  // inclusive scan of run over the block
  unsigned long long inc = run;
  const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
#pragma unroll
  for (int o = 1; o < 32; o <<= 1) {
    unsigned long long v = __shfl_up_sync(0xffffffffu, inc, o);
    if (lane >= o) inc += v;
  }
  if (lane == 31) wsum[wid] = inc;
  __syncthreads();
  if (wid == 0) {
    unsigned long long v = wsum[lane], s = v;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
      unsigned long long u = __shfl_up_sync(0xffffffffu, s, o);
      if (lane >= o) s += u;
    }
    wsum[lane] = s - v;  // exclusive
  }
  __syncthreads();
  unsigned long long pre = wsum[wid] + inc - run;
  if (vec) {
    const float4* w4 = reinterpret_cast<const float4*>(w + lo);
    ulonglong2* C2 = reinterpret_cast<ulonglong2*>(C + lo);
    for (int i = 0; i < ipt / 4; ++i) {
      float4 v = w4[i];
      ulonglong2 c0, c1;
      pre += quantise40(v.x); c0.x = pre;
      pre += quantise40(v.y); c0.y = pre;
      pre += quantise40(v.z); c1.x = pre;
      pre += quantise40(v.w); c1.y = pre;
      C2[2 * i] = c0;
      C2[2 * i + 1] = c1;
    }
  } else {
    for (int i = lo; i < hi; ++i) {
      pre += quantise40(w[i]);
      C[i] = pre;
    }
  }
  if (threadIdx.x == blockDim.x - 1) {
    ctrl->q_total = pre;
    if (pre == 0ull) ctrl->nan_flag = 1;
  }
}

// Large N: two launches.  Blocks of 256 threads x 16 weights; (1) block sums, (2) every block adds
// the sums of the blocks before it (at most 256 of them: N <= 2^20) and scans its own 4096 weights.
constexpr int SCAN_BLOCK = 4096;
__global__ void __launch_bounds__(256)
scan_block_sums_kernel(const float* __restrict__ w, int N, unsigned long long* __restrict__ bsum,
                       const Ctrl* ctrl) {
  __shared__ unsigned long long ws[8];
  if (ctrl->done) return;
  const int base = blockIdx.x * SCAN_BLOCK + threadIdx.x * 16;
  unsigned long long run = 0;
#pragma unroll
  for (int j = 0; j < 16; ++j) run += (base + j < N) ? quantise40(w[base + j]) : 0ull;
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) run += __shfl_xor_sync(0xffffffffu, run, o);
  if ((threadIdx.x & 31) == 0) ws[threadIdx.x >> 5] = run;
  __syncthreads();
  if (threadIdx.x == 0) {
    unsigned long long t = 0;
    for (int k = 0; k < 8; ++k) t += ws[k];
    bsum[blockIdx.x] = t;
  }
}

__global__ void __launch_bounds__(256)
scan_apply_kernel(const float* __restrict__ w, int N, const unsigned long long* __restrict__ bsum,
                  unsigned long long* __restrict__ C, Ctrl* ctrl) {
  __shared__ unsigned long long ws[8];
  __shared__ unsigned long long off_s;
  if (ctrl->done) return;
  const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
  // exclusive prefix of the block sums before this block
  unsigned long long pre = ((int)threadIdx.x < (int)blockIdx.x) ? bsum[threadIdx.x] : 0ull;
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) pre += __shfl_xor_sync(0xffffffffu, pre, o);
  if (lane == 0) ws[wid] = pre;
  __syncthreads();
  if (threadIdx.x == 0) {
    unsigned long long t = 0;
    for (int k = 0; k < 8; ++k) t += ws[k];
    off_s = t;
  }
  __syncthreads();
  const int base = blockIdx.x * SCAN_BLOCK + threadIdx.x * 16;
  unsigned long long q[16], run = 0;
#pragma unroll
  for (int j = 0; j < 16; ++j) { q[j] = (base + j < N) ? quantise40(w[base + j]) : 0ull; run += q[j]; }
  unsigned long long inc = run;
#pragma unroll
  for (int o = 1; o < 32; o <<= 1) {
    unsigned long long v = __shfl_up_sync(0xffffffffu, inc, o);
    if (lane >= o) inc += v;
  }
  __syncthreads();
  if (lane == 31) ws[wid] = inc;
  __syncthreads();
  unsigned long long wpre = 0;
  for (int k = 0; k < wid; ++k) wpre += ws[k];
  unsigned long long acc = off_s + wpre + inc - run;
#pragma unroll
  for (int j = 0; j < 16; ++j) {
    acc += q[j];
    if (base + j < N) C[base + j] = acc;
  }
  if (blockIdx.x == gridDim.x - 1 && threadIdx.x == blockDim.x - 1) {
    ctrl->q_total = acc;
    if (acc == 0ull) ctrl->nan_flag = 1;
  }
}

void launch_quantise_scan(const float* w, int N, unsigned long long* C, Ctrl* ctrl,
                          cudaStream_t st) {
  if (N <= 32768 || N > 256 * SCAN_BLOCK) {
    ++g_launches; launch_pdl(quantise_scan_kernel, 1, 1024, 0, st, w, N, C, ctrl);
    return;
  }
  const int nb = (N + SCAN_BLOCK - 1) / SCAN_BLOCK;
  // block sums live in the pad of C: C has ld = round_up(N,128) entries plus 256 spare (api.cu)
  unsigned long long* sums = C + round_up(N, 128);
  ++g_launches; scan_block_sums_kernel<<<nb, 256, 0, st>>>(w, N, sums, ctrl);
  ++g_launches; scan_apply_kernel<<<nb, 256, 0, st>>>(w, N, sums, C, ctrl);
}

// a_j = #{i : C_i <= t_j}, t_j = floor(((j 2^32 + U) T) / (N 2^32)), clamped to N-1; U = word 0
// of the RESAMPLE stream at the current temperature index.  Once the run is done the map is the
// identity, so that a step enqueued past beta = 1 leaves the particles unchanged.
// flip[j] (NEXT row f4, reading A17): with z2 set, slot j is sign-flipped by the gather iff the top
// bit of word 0 of the Z2 stream at this temperature is set.
__global__ void ancestors_kernel(const unsigned long long* __restrict__ C, int N, uint64_t seed,
                                 int32_t* __restrict__ anc, uint8_t* __restrict__ flip, int z2,
                                 const Ctrl* ctrl) {
  pdl_enter();
  int j = blockIdx.x * blockDim.x + threadIdx.x;
  if (j >= N) return;
  if (ctrl->done || ctrl->q_total == 0ull) { anc[j] = j; flip[j] = 0; return; }
  flip[j] = z2 ? (uint8_t)(philox_draw(seed, TAG_Z2, (uint32_t)ctrl->temp_index, (uint32_t)j, 0u).x >> 31)
               : (uint8_t)0;
  const uint32_t U = philox_draw(seed, TAG_RESAMPLE, (uint32_t)ctrl->temp_index, 0u, 0u).x;
  const unsigned long long T = ctrl->q_total;
  unsigned __int128 num = (unsigned __int128)(((unsigned long long)j << 32) + U) *
                          (unsigned __int128)T;
  unsigned long long tj = (unsigned long long)(num / ((unsigned __int128)((unsigned long long)N << 32)));
  int lo = 0, hi = N;  // first index with C > tj
  while (lo < hi) {
    int mid = (lo + hi) >> 1;
    if (C[mid] <= tj) lo = mid + 1; else hi = mid;
  }
  anc[j] = min(lo, N - 1);
}

void launch_ancestors(const unsigned long long* C, int N, uint64_t seed, int32_t* anc, uint8_t* flip,
                      int z2, Ctrl* ctrl, cudaStream_t st) {
  ++g_launches; launch_pdl(ancestors_kernel, (N + 255) / 256, 256, 0, st, C, N, seed, anc, flip, z2, ctrl);
}

// ---------------------------------------------------------------------------------------------
// P4: phi_out[x][j] = phi_in[x][a_j] (and S, U0).  A thread owns 4 consecutive slots j: four
// scalar gathers (a is monotone, so a warp reads a near-contiguous span) and one 16-byte store
// per site row.  grid.y splits the V rows.  HBM bound: 8 N V bytes.
// ---------------------------------------------------------------------------------------------
constexpr int GATHER_ROWS = 16;
template <bool Z2>
__global__ void __launch_bounds__(256)
gather_kernel(const float* __restrict__ pin, float* __restrict__ pout,
              const float* __restrict__ Sin, float* __restrict__ Sout,
              const float* __restrict__ Uin, float* __restrict__ Uout,
              const int32_t* __restrict__ anc, const uint8_t* __restrict__ flip, int N, int ld,
              int V, Ctrl* ctrl) {
  pdl_enter();
  const int j0 = (blockIdx.x * blockDim.x + threadIdx.x) * 4;
  if (j0 >= ld) return;
  int a[4];
  float sg[4];                        // Z2 flip of the destination slot (S_E, U0 are even in phi)
#pragma unroll
  for (int m = 0; m < 4; ++m) {
    a[m] = (j0 + m < N) ? anc[j0 + m] : -1;
    sg[m] = (Z2 && j0 + m < N && flip[j0 + m]) ? -1.f : 1.f;
  }
  const int x0 = blockIdx.y * GATHER_ROWS, x1 = min(V, x0 + GATHER_ROWS);
  for (int x = x0; x < x1; ++x) {
    const float* src = pin + (size_t)x * ld;
    float4 v;
    v.x = a[0] >= 0 ? src[a[0]] : 0.f;
    v.y = a[1] >= 0 ? src[a[1]] : 0.f;
    v.z = a[2] >= 0 ? src[a[2]] : 0.f;
    v.w = a[3] >= 0 ? src[a[3]] : 0.f;
    if (Z2) { v.x *= sg[0]; v.y *= sg[1]; v.z *= sg[2]; v.w *= sg[3]; }
    *reinterpret_cast<float4*>(pout + (size_t)x * ld + j0) = v;
  }
  if (blockIdx.y == 0) {
    float4 s, u;
    s.x = a[0] >= 0 ? Sin[a[0]] : 0.f; u.x = a[0] >= 0 ? Uin[a[0]] : 0.f;
    s.y = a[1] >= 0 ? Sin[a[1]] : 0.f; u.y = a[1] >= 0 ? Uin[a[1]] : 0.f;
    s.z = a[2] >= 0 ? Sin[a[2]] : 0.f; u.z = a[2] >= 0 ? Uin[a[2]] : 0.f;
    s.w = a[3] >= 0 ? Sin[a[3]] : 0.f; u.w = a[3] >= 0 ? Uin[a[3]] : 0.f;
    *reinterpret_cast<float4*>(Sout + j0) = s;
    *reinterpret_cast<float4*>(Uout + j0) = u;
    // distinct ancestors: a is non-decreasing, count the rises
    int prev = (j0 > 0 && j0 - 1 < N) ? anc[j0 - 1] : -1;
    int cnt = 0;
#pragma unroll
    for (int m = 0; m < 4; ++m)
      if (a[m] >= 0) { cnt += (a[m] != prev); prev = a[m]; }
    unsigned tot = (unsigned)cnt;
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) tot += __shfl_xor_sync(0xffffffffu, tot, o);
    if ((threadIdx.x & 31) == 0 && tot) atomicAdd(&ctrl->n_unique, tot);
  }
}

void launch_gather(const float* phi_in, float* phi_out, const float* S_in, float* S_out,
                   const float* U_in, float* U_out, const int32_t* anc, const uint8_t* flip, int N,
                   int ld, int V, Ctrl* ctrl, cudaStream_t st) {
  // flip == nullptr: no Z2 move (the instantiation without the sign)
  dim3 grid((ld / 4 + 255) / 256, (V + GATHER_ROWS - 1) / GATHER_ROWS);
  ++g_launches;
  if (flip)
    launch_pdl(gather_kernel<true>, grid, 256, 0, st, phi_in, phi_out, S_in, S_out, U_in, U_out, anc, flip, N,
               ld, V, ctrl);
  else
    launch_pdl(gather_kernel<false>, grid, 256, 0, st, phi_in, phi_out, S_in, S_out, U_in, U_out, anc, flip, N,
               ld, V, ctrl);
}

// End of a temperature: record it, advance the index, latch done at beta == 1.
__global__ void finish_step_kernel(Ctrl* ctrl, StepRecord* rec, int max_rec, int k, int N) {
  pdl_enter();
  if (ctrl->done) return;
  int t = ctrl->temp_index;
  if (t < max_rec) {
    StepRecord r;
    r.beta = ctrl->beta; r.delta = ctrl->delta; r.ess_frac = ctrl->ess_frac;
    r.dlogZ = ctrl->dlogZ; r.logZ = ctrl->logZ;
    r.accept_rate = (double)ctrl->n_accept / ((double)k * (double)N);
    r.n_unique = (int)ctrl->n_unique; r.chol_status = ctrl->chol_status;
    r.index = t; r.done = ctrl->beta >= 1.0;
    rec[t] = r;
  }
  ctrl->temp_index = t + 1;
  ctrl->mut_steps += (unsigned long long)k;   // steps enqueued past beta = 1 never get here
  ctrl->n_accept = 0u;
  ctrl->n_unique = 0u;
  if (ctrl->beta >= 1.0) ctrl->done = 1;
}

void launch_finish_step(Ctrl* ctrl, StepRecord* rec, int max_rec, int k, int N, cudaStream_t st) {
  ++g_launches; launch_pdl(finish_step_kernel, 1, 1, 0, st, ctrl, rec, max_rec, k, N);
}

}  // namespace phi4
