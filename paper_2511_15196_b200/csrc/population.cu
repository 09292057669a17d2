// population.cu -- the population step P1-P4: next beta by ESS bisection,
// incremental weights + log Z, exact integer systematic resampling, gather.
#include <cooperative_groups.h>

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

// h(d) = log(a^2 / (b N target)) and h'(d) without FP64 logarithms or divisions: the ratio minus
// one is formed from an FP64 numerator (exact cancellation near the root) and goes through
// log1pf, whose error is relative to h itself; h' only steers the iteration.
__device__ __forceinline__ void ess_h(const EssSums& q, double NT, float& h, float& dh) {
  const double den = q.b * NT;
  const double num = q.a * q.a - den;
  h = log1pf((float)num / (float)den);
  dh = 2.f * (float)q.da / (float)q.a - (float)q.db / (float)q.b;
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
  __shared__ unsigned long long wsum[32];
  float xs[rw::RC];
  int cnt = 0;
  float m = INFINITY;
  // cached layout: thread t owns the contiguous run [t ipt, (t+1) ipt): 16-byte loads and stores
  // when the run is whole and aligned, and the integer scan of P3 is a serial prefix per thread
  // plus ONE warp scan of the run totals
  const int ipt = min(rw::RC, (N + rw::THREADS - 1) / rw::THREADS);
  const int run0 = (int)threadIdx.x * ipt;
  const bool vec = CACHED && (ipt & 3) == 0 && run0 + ipt <= N;
  if (CACHED) {
    cnt = max(0, min(ipt, N - run0));
    if (vec) {
      const float4* s4 = reinterpret_cast<const float4*>(S + run0);
#pragma unroll
      for (int j = 0; j < rw::RC / 4; ++j)
        if (4 * j < ipt) {
          const float4 v = s4[j];
          xs[4 * j] = v.x; xs[4 * j + 1] = v.y; xs[4 * j + 2] = v.z; xs[4 * j + 3] = v.w;
        } else {
          xs[4 * j] = xs[4 * j + 1] = xs[4 * j + 2] = xs[4 * j + 3] = INFINITY;
        }
    } else {
#pragma unroll
      for (int j = 0; j < rw::RC; ++j) xs[j] = j < cnt ? S[run0 + j] : INFINITY;
    }
#pragma unroll
    for (int j = 0; j < rw::RC; ++j) m = fminf(m, xs[j]);
  } else {
    for (int i = threadIdx.x; i < N; i += rw::THREADS) m = fminf(m, S[i]);
  }
  m = warp_min(m);
  if ((threadIdx.x & 31) == 0) smin_s[threadIdx.x >> 5] = m;
  __syncthreads();
  const float smin = warp_min(smin_s[threadIdx.x & 31]);    // every warp reduces the 32 minima
  if (CACHED) {
#pragma unroll
    for (int j = 0; j < rw::RC; ++j) xs[j] -= smin;
  }
  const double beta = ctrl->beta;
  const double rest = 1.0 - beta;
  const double NT = (double)N * (double)ess_target, lN = log((double)N);
  double delta;
  int final_step = 0;
  if (delta_fixed >= 0.0) {
    delta = delta_fixed;
    final_step = (beta + delta >= 1.0);
  } else {
    // thread 0 owns the bracket and the Newton step; the next abscissa and the stop flag go
    // through shared memory
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
        float h, dh;
        ess_h(q, NT, h, dh);
        if (x >= rest && !hi_known) {
          if (h >= 0.f) { stop = 1; fin = 1; xn = rest; }
          hi_known = true;
        }
        if (!stop) {
          if (h > 0.f) lo = x; else hi = x;
          if (fabsf(h) < 1e-9f) stop = 1;
          else {
            xn = x - (double)(h / dh);
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
  const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
  unsigned long long run = 0;
  if (CACHED) {
#pragma unroll
    for (int j = 0; j < rw::RC; ++j)
      if (j < cnt) {
        const float e = expf(-df * xs[j]);
        xs[j] = e;                                   // kept for the scan below
        a += (double)e;
        b += (double)e * (double)e;
        run += quantise40(e);
      }
    if (vec) {
      float4* w4 = reinterpret_cast<float4*>(w + run0);
#pragma unroll
      for (int j = 0; j < rw::RC / 4; ++j)
        if (4 * j < ipt) w4[j] = make_float4(xs[4 * j], xs[4 * j + 1], xs[4 * j + 2], xs[4 * j + 3]);
    } else {
#pragma unroll
      for (int j = 0; j < rw::RC; ++j) if (j < cnt) w[run0 + j] = xs[j];
    }
  } else {
    for (int i = threadIdx.x; i < N; i += rw::THREADS) {
      const float e = expf(-df * (S[i] - smin));
      w[i] = e;
      a += (double)e;
      b += (double)e * (double)e;
    }
  }
  // one round for both block reductions: sum w, sum w^2, and (P3 fused, reading R5) the
  // inclusive integer scan of the run totals q = sum floor(w_i 2^40)
  unsigned long long inc = run;
  if (CACHED && C) {
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
      unsigned long long v = __shfl_up_sync(0xffffffffu, inc, o);
      if (lane >= o) inc += v;
    }
    if (lane == 31) wsum[wid] = inc;
  }
  a = warp_sum(a);
  b = warp_sum(b);
  if (lane == 0) scratch[wid] = make_double4(a, b, 0.0, 0.0);
  __syncthreads();
  {
    double4 t = scratch[lane];                       // every warp reduces the 32 partial sums
    a = warp_sum(t.x);
    b = warp_sum(t.y);
  }
  if (CACHED && C) {
    unsigned long long v = wsum[lane], sc = v;       // ... and scans the 32 warp totals
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
      unsigned long long u = __shfl_up_sync(0xffffffffu, sc, o);
      if (lane >= o) sc += u;
    }
    const unsigned long long warp_off = __shfl_sync(0xffffffffu, sc - v, wid);
    unsigned long long pre = warp_off + inc - run;
    if (vec) {
      ulonglong2* C2 = reinterpret_cast<ulonglong2*>(C + run0);
#pragma unroll
      for (int j = 0; j < rw::RC / 2; ++j)
        if (2 * j < ipt) {
          ulonglong2 c;
          pre += quantise40(xs[2 * j]); c.x = pre;
          pre += quantise40(xs[2 * j + 1]); c.y = pre;
          C2[j] = c;
        }
    } else {
#pragma unroll
      for (int j = 0; j < rw::RC; ++j)
        if (j < cnt) { pre += quantise40(xs[j]); C[run0 + j] = pre; }
    }
    if (threadIdx.x == rw::THREADS - 1) {
      ctrl->q_total = pre;
      if (pre == 0ull) ctrl->nan_flag = 1;
    }
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

// ---------------------------------------------------------------------------------------------
// P1 + P2 (+ the integer scan of P3) for N <= 16384 on a CLUSTER of 8 CTAs.  One CTA holding all
// 16384 actions spends ~2000 cycles per Newton evaluation on instruction issue alone (16 actions
// x 7 instructions x 32 warps on one SM).  Here CTA c of the cluster holds the contiguous chunk
// [c chunk, (c+1) chunk), 8 actions per thread in registers; per evaluation every warp writes
// its four partial sums into the shared memory of ALL eight CTAs (distributed shared memory),
// one cluster barrier, and every thread reduces the 64 partials in the same fixed order and takes
// the Newton step itself: the same numbers in every thread of every CTA, no broadcast.
// Same algorithm (reading R3) and the same stopping rule as next_delta_reweight_body.
// ---------------------------------------------------------------------------------------------
namespace rwc {
constexpr int G = 8, THREADS = 256, WARPS = THREADS / 32, RC = 8, NP = G * WARPS;   // 64 partials
}

__device__ __forceinline__ double4 rwc_reduce64(const double4* slot, int lane) {
  const double4 u = slot[lane], v = slot[lane + 32];
  double4 t = make_double4(u.x + v.x, u.y + v.y, u.z + v.z, u.w + v.w);
  t.x = warp_sum(t.x); t.y = warp_sum(t.y); t.z = warp_sum(t.z); t.w = warp_sum(t.w);
  return t;
}

__global__ void __launch_bounds__(rwc::THREADS)
next_delta_reweight_cluster_kernel(const float* __restrict__ S, int N, float ess_target,
                                   double delta_fixed, float* __restrict__ w,
                                   unsigned long long* __restrict__ C, Ctrl* ctrl) {
  namespace cg = cooperative_groups;
  pdl_enter();
  __shared__ __align__(32) double4 slot[2][rwc::NP];       // partial sums, double-buffered by evaluation
  __shared__ unsigned long long qslot[rwc::NP];            // integer totals of the warps (P3)
  __shared__ float cmin[rwc::G];
  __shared__ float wmin[rwc::WARPS];
  if (ctrl->done) return;                                  // (uniform over the cluster)
  cg::cluster_group cluster = cg::this_cluster();
  const int rank = (int)cluster.block_rank();
  const int tid = threadIdx.x, lane = tid & 31, wid = tid >> 5;
  const int ipt = (N + rwc::G * rwc::THREADS - 1) / (rwc::G * rwc::THREADS);      // <= 8
  const int run0 = (rank * rwc::THREADS + tid) * ipt;
  const int cnt = max(0, min(ipt, N - run0));
  const bool vec = (ipt & 3) == 0 && run0 + ipt <= N;
  float xs[rwc::RC];
  if (vec) {
    const float4* s4 = reinterpret_cast<const float4*>(S + run0);
#pragma unroll
    for (int j = 0; j < rwc::RC / 4; ++j)
      if (4 * j < ipt) {
        const float4 v = s4[j];
        xs[4 * j] = v.x; xs[4 * j + 1] = v.y; xs[4 * j + 2] = v.z; xs[4 * j + 3] = v.w;
      } else {
        xs[4 * j] = xs[4 * j + 1] = xs[4 * j + 2] = xs[4 * j + 3] = INFINITY;
      }
  } else {
#pragma unroll
    for (int j = 0; j < rwc::RC; ++j) xs[j] = j < cnt ? S[run0 + j] : INFINITY;
  }
  float m = INFINITY;
#pragma unroll
  for (int j = 0; j < rwc::RC; ++j) m = fminf(m, xs[j]);
  m = warp_min(m);
  if (lane == 0) wmin[wid] = m;
  __syncthreads();
  if (tid < rwc::G) {                                      // thread g: this CTA's minimum to CTA g
    float v = wmin[0];
#pragma unroll
    for (int k = 1; k < rwc::WARPS; ++k) v = fminf(v, wmin[k]);
    *cluster.map_shared_rank(&cmin[rank], tid) = v;
  }
  cluster.sync();
  float smin = cmin[0];
#pragma unroll
  for (int g = 1; g < rwc::G; ++g) smin = fminf(smin, cmin[g]);
#pragma unroll
  for (int j = 0; j < rwc::RC; ++j) xs[j] -= smin;

  const double beta = ctrl->beta;
  const double rest = 1.0 - beta;
  const double NT = (double)N * (double)ess_target, lN = log((double)N);
  double delta;
  int final_step = 0;
  int par = 0;
  if (delta_fixed >= 0.0) {
    delta = delta_fixed;
    final_step = (beta + delta >= 1.0);
  } else {
    double lo = 0.0, hi = rest;
    bool hi_known = false;
    const double prev = ctrl->delta;
    double x = (prev > 0.0 && prev < rest) ? prev : rest;
    delta = rest;
    for (int it = 0; it < 64; ++it) {
      const float df = (float)x * 1.4426950408889634f;
      float a = 0.f, b = 0.f, da = 0.f, db = 0.f;
#pragma unroll
      for (int j = 0; j < rwc::RC; ++j)
        if (j < cnt) {
          float e;
          asm("ex2.approx.ftz.f32 %0, %1;" : "=f"(e) : "f"(-df * xs[j]));
          const float e2 = e * e;
          a += e; b += e2;
          da = fmaf(xs[j], e, da); db = fmaf(xs[j], e2, db);
        }
      double4 t = make_double4(warp_sum((double)a), warp_sum((double)b), warp_sum((double)da),
                               warp_sum((double)db));
      if (lane < rwc::G) *cluster.map_shared_rank(&slot[par][rank * rwc::WARPS + wid], lane) = t;
      cluster.sync();
      t = rwc_reduce64(slot[par], lane);
      par ^= 1;
      EssSums q{t.x, t.y, -t.z, -2.0 * t.w};
      int stop = 0, fin = 0;
      double xn = x;
      float h, dh;
      ess_h(q, NT, h, dh);
      if (x >= rest && !hi_known) {
        if (h >= 0.f) { stop = 1; fin = 1; xn = rest; }
        hi_known = true;
      }
      if (!stop) {
        if (h > 0.f) lo = x; else hi = x;
        if (fabsf(h) < 1e-9f) stop = 1;
        else {
          xn = x - (double)(h / dh);
          if (!(xn > lo && xn < hi)) {
            if (!hi_known && xn >= hi) xn = rest;
            else if (hi_known) xn = 0.5 * (lo + hi);
            else xn = fmin(rest, 2.0 * x);
          }
          if (fabs(xn - x) <= 1e-7 * xn && !(xn >= rest && !hi_known)) stop = 1;
        }
      }
      x = xn;
      delta = x;
      final_step = fin;
      if (stop) break;
    }
  }
  // P2: weights, their sums, and (P3, reading R5) the integer scan of q_i = floor(w_i 2^40)
  const float df = (float)delta;
  double a = 0.0, b = 0.0;
  unsigned long long run = 0;
#pragma unroll
  for (int j = 0; j < rwc::RC; ++j)
    if (j < cnt) {
      const float e = expf(-df * xs[j]);
      xs[j] = e;
      a += (double)e;
      b += (double)e * (double)e;
      run += quantise40(e);
    }
  if (vec) {
    float4* w4 = reinterpret_cast<float4*>(w + run0);
#pragma unroll
    for (int j = 0; j < rwc::RC / 4; ++j)
      if (4 * j < ipt) w4[j] = make_float4(xs[4 * j], xs[4 * j + 1], xs[4 * j + 2], xs[4 * j + 3]);
  } else {
#pragma unroll
    for (int j = 0; j < rwc::RC; ++j) if (j < cnt) w[run0 + j] = xs[j];
  }
  unsigned long long inc = run;
#pragma unroll
  for (int o = 1; o < 32; o <<= 1) {
    unsigned long long v = __shfl_up_sync(0xffffffffu, inc, o);
    if (lane >= o) inc += v;
  }
  const unsigned long long wtot = __shfl_sync(0xffffffffu, inc, 31);
  {
    const double4 t = make_double4(warp_sum(a), warp_sum(b), 0.0, 0.0);
    const int me = rank * rwc::WARPS + wid;
    if (lane < rwc::G) {
      *cluster.map_shared_rank(&slot[par][me], lane) = t;
      *cluster.map_shared_rank(&qslot[me], lane) = wtot;
    }
  }
  cluster.sync();
  {
    const double4 t = rwc_reduce64(slot[par], lane);
    a = t.x; b = t.y;
  }
  if (C) {
    // exclusive prefix of the 64 warp totals at this warp's position (warps are numbered in
    // element order: rank-major), then the serial prefix inside the thread's run
    const int me = rank * rwc::WARPS + wid;
    const unsigned long long q0 = qslot[lane], q1 = qslot[lane + 32];
    unsigned long long part = (lane < me ? q0 : 0ull) + (lane + 32 < me ? q1 : 0ull);
    unsigned long long tot = q0 + q1;
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) {
      part += __shfl_xor_sync(0xffffffffu, part, o);
      tot += __shfl_xor_sync(0xffffffffu, tot, o);
    }
    unsigned long long pre = part + inc - run;
    if (vec) {
      ulonglong2* C2 = reinterpret_cast<ulonglong2*>(C + run0);
#pragma unroll
      for (int j = 0; j < rwc::RC / 2; ++j)
        if (2 * j < ipt) {
          ulonglong2 c;
          pre += quantise40(xs[2 * j]); c.x = pre;
          pre += quantise40(xs[2 * j + 1]); c.y = pre;
          C2[j] = c;
        }
    } else {
#pragma unroll
      for (int j = 0; j < rwc::RC; ++j)
        if (j < cnt) { pre += quantise40(xs[j]); C[run0 + j] = pre; }
    }
    if (rank == 0 && tid == 0) {
      ctrl->q_total = tot;
      if (tot == 0ull) ctrl->nan_flag = 1;
    }
  }
  if (rank == 0 && tid == 0) {
    double dlz = -delta * (double)smin + log(a) - lN;
    ctrl->delta = delta;
    ctrl->beta = final_step ? 1.0 : beta + delta;
    ctrl->ess_frac = a * a / (b * (double)N);
    ctrl->dlogZ = dlz;
    ctrl->logZ += dlz;
    ctrl->S_min = smin;
    if (!isfinite(dlz)) ctrl->nan_flag = 1;
  }
  cluster.sync();          // no CTA exits while another may still write into its shared memory
}

template <typename... KArgs, typename... Args>
static cudaError_t launch_pdl_cluster(void (*kernel)(KArgs...), int cluster, int threads, cudaStream_t st,
                                      Args&&... args) {
  cudaLaunchConfig_t cfg = {};
  cfg.gridDim = dim3(cluster); cfg.blockDim = dim3(threads); cfg.dynamicSmemBytes = 0; cfg.stream = st;
  cudaLaunchAttribute at[2];
  at[0].id = cudaLaunchAttributeClusterDimension;
  at[0].val.clusterDim.x = cluster; at[0].val.clusterDim.y = 1; at[0].val.clusterDim.z = 1;
  at[1].id = cudaLaunchAttributeProgrammaticStreamSerialization;
  at[1].val.programmaticStreamSerializationAllowed = 1;
  cfg.attrs = at;
  cfg.numAttrs = pdl_enabled() ? 2 : 1;
  return cudaLaunchKernelEx(&cfg, kernel, KArgs(args)...);
}

// C != nullptr and N <= 16384: the integer scan of P3 runs in the same kernel (the weights are
// still in registers); returns whether it did, so that the caller can skip launch_quantise_scan.
bool launch_next_delta_reweight(const float* S, int N, float ess_target, double delta_fixed,
                                float* w, unsigned long long* C, Ctrl* ctrl, cudaStream_t st) {
  const bool fused = C != nullptr && N <= rw::THREADS * rw::RC;
  ++g_launches;
  if (N <= rwc::G * rwc::THREADS * rwc::RC) {
    launch_pdl_cluster(next_delta_reweight_cluster_kernel, rwc::G, rwc::THREADS, st, S, N, ess_target,
                       delta_fixed, w, C, ctrl);
    return fused;
  }
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
// t_j exactly, without a 128-bit division: (P T) >> 32 is a 74-bit number (P < 2^49, T < 2^57);
// long division by N in base 2^32 (N < 2^21, so every partial remainder fits 64 bits).
__device__ __forceinline__ unsigned long long resample_threshold(int j, uint32_t U, unsigned long long T,
                                                                 int N) {
  const unsigned long long P = ((unsigned long long)j << 32) + U;
  const unsigned long long lo = P * T, hi = __umul64hi(P, T);
  const unsigned long long x2 = hi >> 32, x1 = hi & 0xffffffffull, x0 = lo >> 32;
  const unsigned long long n = (unsigned long long)N;
  unsigned long long r = x2 % n;                    // (x2 / n = 0: t_j < T < 2^64)
  r = (r << 32) + x1;
  const unsigned long long q1 = r / n;
  r = ((r % n) << 32) + x0;
  return (q1 << 32) + r / n;
}

__device__ __forceinline__ uint8_t z2_flip_of(uint64_t seed, const Ctrl* ctrl, int j, int z2) {
  if (!z2 || ctrl->done || ctrl->q_total == 0ull) return 0;
  return (uint8_t)(philox_draw(seed, TAG_Z2, (uint32_t)ctrl->temp_index, (uint32_t)j, 0u).x >> 31);
}

// Two-level search: the block first reads 256 samples of the CDF (the last entry of each of 256
// equal segments: one round trip to L2), every thread finds its segment in shared memory and
// finishes inside it -- log2(N / 256) dependent global loads instead of log2(N).
__global__ void __launch_bounds__(256)
ancestors_kernel(const unsigned long long* __restrict__ C, int N, uint64_t seed,
                 int32_t* __restrict__ anc, uint8_t* __restrict__ flip, int z2, const Ctrl* ctrl) {
  pdl_enter();
  __shared__ unsigned long long samp[256];
  const int j = blockIdx.x * blockDim.x + threadIdx.x;
  const unsigned long long T = ctrl->q_total;
  if (ctrl->done || T == 0ull) {                   // (block-uniform) identity map
    if (j < N) { anc[j] = j; flip[j] = 0; }
    return;
  }
  const int seg = (N + 255) >> 8;                   // entries per segment
  {
    const long long e = (long long)(threadIdx.x + 1) * seg - 1;
    samp[threadIdx.x] = C[e < N ? e : N - 1];
  }
  __syncthreads();
  if (j >= N) return;
  const uint32_t U = philox_draw(seed, TAG_RESAMPLE, (uint32_t)ctrl->temp_index, 0u, 0u).x;
  const unsigned long long t = resample_threshold(j, U, T, N);
  int s0 = 0, s1 = 255;                             // first segment whose last entry is > t (one exists:
                                                    // t < T): 256 outcomes, eight halvings
#pragma unroll
  for (int step = 0; step < 8; ++step) {
    const int mid = (s0 + s1) >> 1;
    if (samp[mid] <= t) s0 = mid + 1; else s1 = mid;
  }
  int lo = min(N, s0 * seg), hi = min(N, lo + seg);  // first index with C > t lies in [lo, hi]
  for (int span = seg; span > 0; span >>= 1) {
    const int mid = (lo + hi) >> 1;
    if (lo < hi) {
      if (C[mid] <= t) lo = mid + 1; else hi = mid;
    }
  }
  anc[j] = min(lo, N - 1);
  flip[j] = z2_flip_of(seed, ctrl, j, z2);
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
__global__ void finish_step_kernel(Ctrl* ctrl, StepRecord* rec, int max_rec, int k, int N, HostPoll* hp) {
  pdl_enter();
  if (ctrl->done) return;
  finish_step_device(ctrl, rec, max_rec, k, N, hp);
}

void launch_finish_step(Ctrl* ctrl, StepRecord* rec, int max_rec, int k, int N, HostPoll* hp, cudaStream_t st) {
  ++g_launches; launch_pdl(finish_step_kernel, 1, 1, 0, st, ctrl, rec, max_rec, k, N, hp);
}

}  // namespace phi4
