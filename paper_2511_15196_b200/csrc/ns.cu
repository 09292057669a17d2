// ns.cu -- nested-sampling population step N1-N4 (PAPER.md:53(iv), :161, :170, :174; readings
// A5, A6; volume bookkeeping after Skilling 2006, PAPER.md:141 ref [37]).
#include "kernels.cuh"
#include "philox.cuh"

namespace phi4 {

__device__ __forceinline__ double logaddexp_d(double a, double b) {
  if (a == -INFINITY) return b;
  if (b == -INFINITY) return a;
  double m = fmax(a, b);
  return m + log(exp(a - m) + exp(b - m));
}

// Bitonic network on 64-bit composite keys (descending S_E, ascending index; pad keys sort last).
// A block of 1024 threads holds 1024 E keys, thread t the keys t E .. t E + E - 1 in registers:
// partners inside the thread are exchanged in registers, partners inside the warp by shuffles,
// and only the strides that cross warps (j >= 32 E) go through shared memory -- 15 of the 78
// stages at n = 4096 instead of a barrier after every stage.
__device__ __forceinline__ unsigned long long ns_key(float S, int i) {
  const uint32_t b = __float_as_uint(S);
  const uint32_t asc = (b & 0x80000000u) ? ~b : (b | 0x80000000u);   // ascending-orderable
  return ((unsigned long long)(~asc) << 32) | (uint32_t)i;           // descending S, ascending i
}

// The strides jstart, jstart / 2, ..., 1 of merge stage k for the block's 1024 E keys, whose global
// positions start at `base` (a multiple of 1024 E): position gi sorts ascending iff (gi & k) == 0.
template <int E>
__device__ __forceinline__ void bitonic_strides(unsigned long long (&kr)[E], unsigned long long* keys,
                                                int k, int jstart, int base) {
  const int tid = threadIdx.x;
  for (int j = jstart; j >= E && j > 0; j >>= 1) {
    if (j >= 32 * E) {
      // partner in another warp: through shared memory
#pragma unroll
      for (int e = 0; e < E; ++e) keys[tid * E + e] = kr[e];
      __syncthreads();
#pragma unroll
      for (int e = 0; e < E; ++e) {
        const int i = tid * E + e;
        const unsigned long long y = keys[i ^ j];
        const bool keep_min = ((i & j) == 0) == (((base + i) & k) == 0);
        kr[e] = keep_min ? (kr[e] < y ? kr[e] : y) : (kr[e] > y ? kr[e] : y);
      }
      __syncthreads();
    } else {
      // partner in another lane of this warp, same register slot
      const int lm = j / E;
#pragma unroll
      for (int e = 0; e < E; ++e) {
        const int i = tid * E + e;
        const unsigned long long y = __shfl_xor_sync(0xffffffffu, kr[e], lm);
        const bool keep_min = ((i & j) == 0) == (((base + i) & k) == 0);
        kr[e] = keep_min ? (kr[e] < y ? kr[e] : y) : (kr[e] > y ? kr[e] : y);
      }
    }
  }
  // partners inside this thread: strides E/2 .. 1 (compile-time register indices)
#pragma unroll
  for (int jj = E >> 1; jj > 0; jj >>= 1) {
    if (jj <= jstart) {
#pragma unroll
      for (int e = 0; e < E; ++e) {
        if ((e & jj) == 0) {
          const int i = tid * E + e;
          const bool up = ((base + i) & k) == 0;
          const unsigned long long x = kr[e], y = kr[e | jj];
          if ((x > y) == up) { kr[e] = y; kr[e | jj] = x; }
        }
      }
    }
  }
}

// Full sort of the block's 1024 E keys (built from S; positions >= n are pad keys); the sorted keys
// end in `keys` (shared memory).
template <int E>
__device__ __forceinline__ void bitonic_sort_block(const float* __restrict__ S, int n,
                                                   unsigned long long* keys, int base = 0) {
  const int tid = threadIdx.x, NP = 1024 * E;
  unsigned long long kr[E];
#pragma unroll
  for (int e = 0; e < E; ++e) {
    const int i = base + tid * E + e;
    kr[e] = i < n ? ns_key(S[i], i) : ~0ull;
  }
  for (int k = 2; k <= NP; k <<= 1) bitonic_strides<E>(kr, keys, k, k >> 1, base);
#pragma unroll
  for (int e = 0; e < E; ++e) keys[tid * E + e] = kr[e];
  __syncthreads();
}

// The kd smallest keys (= the dead points) of the block's 1024 E keys, sorted, without sorting the
// rest: radix select of the kd-th smallest key (8 bits per pass from the top; the keys are distinct,
// so at the latest the eighth pass isolates it; the pass stops as soon as a whole bin is taken),
// compaction of the selected keys, and a 1024-key bitonic sort of those.  For kd <= 1024.
template <int E>
__device__ __forceinline__ void topk_sort_block(const float* __restrict__ S, int n, int kd,
                                                unsigned long long* keys) {
  __shared__ int hist[256];
  __shared__ int sel_digit, sel_before, sel_all;
  __shared__ int wcnt[32];
  const int tid = threadIdx.x, lane = tid & 31, wid = tid >> 5;
  unsigned long long kr[E];
#pragma unroll
  for (int e = 0; e < E; ++e) {
    const int i = tid * E + e;
    kr[e] = i < n ? ns_key(S[i], i) : ~0ull;
  }
  unsigned long long prefix = 0ull, mask = 0ull;
  int remaining = kd;                                    // rank of the threshold among the candidates
  for (int pass = 0; pass < 8; ++pass) {
    const int shift = 56 - 8 * pass;
    if (tid < 256) hist[tid] = 0;
    __syncthreads();
#pragma unroll
    for (int e = 0; e < E; ++e)
      if ((kr[e] & mask) == prefix) atomicAdd(&hist[(int)((kr[e] >> shift) & 255ull)], 1);
    __syncthreads();
    if (wid == 0) {
      // lane l: bins 8 l .. 8 l + 7; find the bin that holds rank `remaining`
      int c[8], tot = 0;
#pragma unroll
      for (int b = 0; b < 8; ++b) { c[b] = hist[8 * lane + b]; tot += c[b]; }
      int inc = tot;
#pragma unroll
      for (int o = 1; o < 32; o <<= 1) {
        const int v = __shfl_up_sync(0xffffffffu, inc, o);
        if (lane >= o) inc += v;
      }
      int before = inc - tot;                            // candidates in the bins of lower lanes
      if (before < remaining && remaining <= inc) {      // exactly one lane
        int b = 0;
        while (before + c[b] < remaining) { before += c[b]; ++b; }
        sel_digit = 8 * lane + b;
        sel_before = before;
        sel_all = (remaining - before == c[b]);          // the whole bin is taken: done
      }
    }
    __syncthreads();
    prefix |= (unsigned long long)sel_digit << shift;
    mask |= 255ull << shift;
    remaining -= sel_before;
    if (sel_all) break;
  }
  // selected: (key & mask) <= prefix -- exactly kd keys; compact them in index order of the threads
  int cnt = 0;
#pragma unroll
  for (int e = 0; e < E; ++e) cnt += ((kr[e] & mask) <= prefix) ? 1 : 0;
  int inc = cnt;
#pragma unroll
  for (int o = 1; o < 32; o <<= 1) {
    const int v = __shfl_up_sync(0xffffffffu, inc, o);
    if (lane >= o) inc += v;
  }
  if (lane == 31) wcnt[wid] = inc;
  __syncthreads();
  if (wid == 0) {
    const int v = wcnt[lane];
    int sc = v;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
      const int u = __shfl_up_sync(0xffffffffu, sc, o);
      if (lane >= o) sc += u;
    }
    wcnt[lane] = sc - v;
  }
  __syncthreads();
  int pos = wcnt[wid] + inc - cnt;
#pragma unroll
  for (int e = 0; e < E; ++e)
    if ((kr[e] & mask) <= prefix) keys[pos++] = kr[e];
  __syncthreads();
  // sort the kd selected keys (padded to 1024 with keys that sort last)
  unsigned long long k1[1];
  k1[0] = tid < kd ? keys[tid] : ~0ull;
  __syncthreads();
  for (int k = 2; k <= 1024; k <<= 1) bitonic_strides<1>(k1, keys, k, k >> 1, 0);
  keys[tid] = k1[0];
  __syncthreads();
}

// ---- more than 16384 live points: the same network across blocks, keys in global memory --------
constexpr int NS_BLOCK_KEYS = 16384;
__global__ void __launch_bounds__(1024)
ns_sort_local_kernel(const float* __restrict__ S, int n, unsigned long long* __restrict__ gkeys,
                     const Ctrl* ctrl) {
  extern __shared__ unsigned long long keys[];
  if (ctrl->done) return;
  const int base = blockIdx.x * NS_BLOCK_KEYS;
  bitonic_sort_block<16>(S, n, keys, base);
  for (int i = threadIdx.x; i < NS_BLOCK_KEYS; i += blockDim.x) gkeys[base + i] = keys[i];
}
// one stride j >= 16384 of merge stage k: thread = the lower element of a pair
__global__ void ns_merge_global_kernel(unsigned long long* __restrict__ gkeys, int j, int k, int np2,
                                       const Ctrl* ctrl) {
  if (ctrl->done) return;
  const int t = blockIdx.x * blockDim.x + threadIdx.x;
  if (t >= np2 / 2) return;
  const int i = ((t & ~(j - 1)) << 1) | (t & (j - 1));          // bit j clear
  const unsigned long long x = gkeys[i], y = gkeys[i | j];
  const bool up = (i & k) == 0;
  if ((x > y) == up) { gkeys[i] = y; gkeys[i | j] = x; }
}
// the strides 8192 .. 1 of merge stage k, block-local
__global__ void __launch_bounds__(1024)
ns_merge_local_kernel(unsigned long long* __restrict__ gkeys, int k, const Ctrl* ctrl) {
  extern __shared__ unsigned long long keys[];
  if (ctrl->done) return;
  const int base = blockIdx.x * NS_BLOCK_KEYS, tid = threadIdx.x;
  unsigned long long kr[16];
#pragma unroll
  for (int e = 0; e < 16; ++e) kr[e] = gkeys[base + tid * 16 + e];
  bitonic_strides<16>(kr, keys, k, NS_BLOCK_KEYS >> 1, base);
#pragma unroll
  for (int e = 0; e < 16; ++e) gkeys[base + tid * 16 + e] = kr[e];
}

// N1 + N2 + survivors + start choice in one CTA.
//  N1: 64-bit keys (descending S_E, ascending index) bitonic-sorted in shared memory; the first
//      k_del are the dead points, S_star = smallest S_E among them.
//  N2: logX_j = logX_{j-1} - 1/(n-j+1), w_j = X_{j-1} - X_j, Z += w_j e^{-S_j}; the logX offsets
//      do not depend on the data, so the batch is one parallel log-sum-exp.
//  N3 (choice): survivors in index order by a flag scan; walker j starts from survivor number
//      (word0 mod (n - k_del)) of Philox stream NS_START (c1 = j, c2 = iteration).
// More than 16384 live points: the keys arrive sorted in global memory (a.gkeys, multi-block
// network above) and the survivor flags live in global memory too (a.gflag).
__global__ void __launch_bounds__(1024)
ns_select_evidence_kernel(NsArgs a) {
  pdl_enter();
  extern __shared__ unsigned long long skeys[];  // npow2 keys; later reused as int flags
  __shared__ double scratch[33];
  __shared__ int wsum[32];
  Ctrl* ctrl = a.ctrl;
  if (ctrl->done) return;
  const int n = a.n, kd = a.k_del, tid = threadIdx.x, nt = blockDim.x;
  const bool big = n > NS_BLOCK_KEYS;
  const unsigned long long* keys = big ? a.gkeys : skeys;
  if (!big) {
    int np2 = 1024;                  // padded to the block: thread t holds keys t E .. t E + E - 1
    while (np2 < n) np2 <<= 1;
    if (kd <= 1024 && 4 * kd <= n) {
      // few dead points: select them, sort only them (the order of the survivors is never used)
      switch (np2 >> 10) {
        case 1: topk_sort_block<1>(a.S, n, kd, skeys); break;
        case 2: topk_sort_block<2>(a.S, n, kd, skeys); break;
        case 4: topk_sort_block<4>(a.S, n, kd, skeys); break;
        case 8: topk_sort_block<8>(a.S, n, kd, skeys); break;
        default: topk_sort_block<16>(a.S, n, kd, skeys); break;
      }
    } else {
      switch (np2 >> 10) {
        case 1: bitonic_sort_block<1>(a.S, n, skeys); break;
        case 2: bitonic_sort_block<2>(a.S, n, skeys); break;
        case 4: bitonic_sort_block<4>(a.S, n, skeys); break;
        case 8: bitonic_sort_block<8>(a.S, n, skeys); break;
        default: bitonic_sort_block<16>(a.S, n, skeys); break;
      }
    }
  }
  const int it = ctrl->temp_index;
  const double logX0 = ctrl->logX;
  // dead list, threshold
  for (int j = tid; j < kd; j += nt) a.dead[j] = (int)(uint32_t)keys[j];
  const float S_star = a.S[(int)(uint32_t)keys[kd - 1]];
  // evidence of the batch: two passes (max, then sum) over the dead points, k_del / 1024 per thread
  double best = -INFINITY;
  for (int j = tid; j < kd; j += nt) {
    const double lx = logX0 - a.hsum[j];                                  // logX_{j'-1}, j' = j+1
    const double logw = lx + a.hsum[kd + 1 + j];                          // + log(1 - e^{-1/(n-j'+1)})
    const int d = (int)(uint32_t)keys[j];
    const float Sd = a.S[d];
    if (it < a.max_iters) {
      const size_t slot = (size_t)it * kd + j;
      a.dead_S[slot] = Sd;
      a.dead_logw[slot] = logw;
    }
    best = fmax(best, logw - (double)Sd);
  }
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) best = fmax(best, __shfl_xor_sync(0xffffffffu, best, o));
  if ((tid & 31) == 0) scratch[tid >> 5] = best;
  __syncthreads();
  if (tid == 0) {
    double m = -INFINITY;
    for (int k = 0; k < (nt >> 5); ++k) m = fmax(m, scratch[k]);
    scratch[32] = m;
  }
  __syncthreads();
  best = scratch[32];
  double e = 0.0;
  for (int j = tid; j < kd; j += nt) {
    const double logw = logX0 - a.hsum[j] + a.hsum[kd + 1 + j];
    e += exp(logw - (double)a.S[(int)(uint32_t)keys[j]] - best);
  }
  e = block_sum(e, scratch);
  __syncthreads();
  // survivors: flags over n, contiguous run per thread, block scan
  // (the dead indices were written to a.dead above: the keys' storage becomes the flag array)
  int* flags = big ? a.gflag : reinterpret_cast<int*>(skeys);
  __syncthreads();
  for (int i = tid; i < n; i += nt) flags[i] = 1;
  __syncthreads();
  for (int j = tid; j < kd; j += nt) flags[a.dead[j]] = 0;
  __syncthreads();
  const int ipt = (n + nt - 1) / nt;
  const int lo = min(n, tid * ipt), hi = min(n, lo + ipt);
  int run = 0;
  for (int i = lo; i < hi; ++i) run += flags[i];
  int inc = run;
  const int lane = tid & 31, wid = tid >> 5;
#pragma unroll
  for (int o = 1; o < 32; o <<= 1) {
    int v = __shfl_up_sync(0xffffffffu, inc, o);
    if (lane >= o) inc += v;
  }
  if (lane == 31) wsum[wid] = inc;
  __syncthreads();
  if (wid == 0) {
    int v = wsum[lane], s = v;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
      int u = __shfl_up_sync(0xffffffffu, s, o);
      if (lane >= o) s += u;
    }
    wsum[lane] = s - v;
  }
  __syncthreads();
  int pos = wsum[wid] + inc - run;
  for (int i = lo; i < hi; ++i)
    if (flags[i]) a.surv[pos++] = i;
  __syncthreads();
  __threadfence_block();
  const int ns = n - kd;
  for (int j = tid; j < kd; j += nt) {
    uint32_t r = philox_draw(a.seed, TAG_NS_START, (uint32_t)it, (uint32_t)j, 0u).x;
    a.start[j] = a.surv[r % (uint32_t)ns];
  }
  if (tid == 0) {
    ctrl->logX = logX0 - a.hsum[kd];
    ctrl->logZ = logaddexp_d(ctrl->logZ, best + log(e));
    ctrl->S_star = (double)S_star;
  }
}

size_t ns_sort_scratch_keys(int n) {          // global keys of the multi-block sort (0: not needed)
  if (n <= NS_BLOCK_KEYS) return 0;
  size_t np2 = NS_BLOCK_KEYS;
  while (np2 < (size_t)n) np2 <<= 1;
  return np2;
}

void launch_ns_select_evidence(const NsArgs& a, cudaStream_t st) {
  static bool attr_done = false;
  const int kb = NS_BLOCK_KEYS * (int)sizeof(unsigned long long);
  if (!attr_done) {
    cudaFuncSetAttribute(ns_select_evidence_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, kb);
    cudaFuncSetAttribute(ns_sort_local_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, kb);
    cudaFuncSetAttribute(ns_merge_local_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, kb);
    attr_done = true;
  }
  if (a.n <= NS_BLOCK_KEYS) {
    int np2 = 1024;
    while (np2 < a.n) np2 <<= 1;
    ++g_launches;
    launch_pdl(ns_select_evidence_kernel, 1, 1024, (size_t)np2 * sizeof(unsigned long long), st, a);
    return;
  }
  // multi-block bitonic network: block-local sorts of 16384 keys, then per merge stage k the
  // strides >= 16384 one launch each over global memory and the rest block-local
  const int np2 = (int)ns_sort_scratch_keys(a.n), nb = np2 / NS_BLOCK_KEYS;
  ++g_launches; ns_sort_local_kernel<<<nb, 1024, kb, st>>>(a.S, a.n, a.gkeys, a.ctrl);
  for (int k = 2 * NS_BLOCK_KEYS; k <= np2; k <<= 1) {
    for (int j = k >> 1; j >= NS_BLOCK_KEYS; j >>= 1) {
      ++g_launches; ns_merge_global_kernel<<<np2 / 2 / 256, 256, 0, st>>>(a.gkeys, j, k, np2, a.ctrl);
    }
    ++g_launches; ns_merge_local_kernel<<<nb, 1024, kb, st>>>(a.gkeys, k, a.ctrl);
  }
  ++g_launches; ns_select_evidence_kernel<<<1, 1024, 0, st>>>(a);
}

// hsum[j] = sum_{m=1..j} 1/(n-m+1), j = 0..k_del: the data-independent volume shrinkage of
// reading A6, tabulated once at ns_init.
__global__ void ns_hsum_kernel(double* hsum, int n, int k_del) {
  // second table (data-independent, so once and not per iteration: an FP64 exp and log1p per dead point):
  // hsum[k_del + 1 + j] = log(1 - e^{-1/(n-j)}), the log width factor of dead point j
  for (int j = threadIdx.x; j < k_del; j += blockDim.x)
    hsum[k_del + 1 + j] = log1p(-exp(-1.0 / (double)(n - j)));
  if (threadIdx.x != 0) return;
  double acc = 0.0;
  hsum[0] = 0.0;
  for (int m = 1; m <= k_del; ++m) { acc += 1.0 / (double)(n - m + 1); hsum[m] = acc; }
}
void launch_ns_hsum(double* hsum, int n, int k_del, cudaStream_t st) {
  ++g_launches; ns_hsum_kernel<<<1, 256, 0, st>>>(hsum, n, k_del);
}

// N3 gather: walker j <- live point start[j].  One thread per (site, walker): the walker index is
// the fast one, so the stores are coalesced and the gathers hit 512 distinct columns of one row.
__global__ void ns_load_walkers_kernel(NsArgs a) {
  pdl_enter();
  if (a.ctrl->done) return;
  const int j = blockIdx.x * blockDim.x + threadIdx.x;
  const int x = blockIdx.y;
  if (j >= a.ldw) return;
  const bool live = j < a.k_del;
  const int src = live ? a.start[j] : 0;
  a.wphi[(size_t)x * a.ldw + j] = live ? a.phi[(size_t)x * a.ld + src] : 0.f;
  if (x == 0) {
    a.wS[j] = live ? a.S[src] : 0.f;
    a.wU[j] = live ? a.U0[src] : 0.f;
  }
}

// Magnetisation of the dead points (logged for the posterior observables): one warp per point.
__global__ void ns_dead_M_kernel(NsArgs a) {
  pdl_enter();
  if (a.ctrl->done) return;
  const int j = (blockIdx.x * blockDim.x + threadIdx.x) >> 5, lane = threadIdx.x & 31;
  if (j >= a.k_del) return;
  const int d = a.dead[j];
  float m = 0.f;
  for (int x = lane; x < a.V; x += 32) m += a.phi[(size_t)x * a.ld + d];
  m = warp_sum(m);
  const int it = a.ctrl->temp_index;
  if (lane == 0 && it < a.max_iters) a.dead_M[(size_t)it * a.k_del + j] = m / (float)a.V;
}

void launch_ns_load_walkers(const NsArgs& a, cudaStream_t st) {
  ++g_launches; launch_pdl(ns_dead_M_kernel, (a.k_del * 32 + 127) / 128, 128, 0, st, a);
  dim3 grid((a.ldw + 127) / 128, a.V);
  ++g_launches; launch_pdl(ns_load_walkers_kernel, grid, 128, 0, st, a);
}

// N3 scatter: dead slot dead[j] <- walker j, one thread per (site, walker).
__global__ void ns_store_walkers_kernel(NsArgs a) {
  pdl_enter();
  if (a.ctrl->done) return;
  const int j = blockIdx.x * blockDim.x + threadIdx.x;
  const int x = blockIdx.y;
  if (j >= a.k_del) return;
  const int d = a.dead[j];
  a.phi[(size_t)x * a.ld + d] = a.wphi[(size_t)x * a.ldw + j];
  if (x == 0) {
    a.S[d] = a.wS[j];
    a.U0[d] = a.wU[j];
  }
}

void launch_ns_store_walkers(const NsArgs& a, cudaStream_t st) {
  dim3 grid((a.k_del + 127) / 128, a.V);
  ++g_launches; launch_pdl(ns_store_walkers_kernel, grid, 128, 0, st, a);
}

// N4: remaining = X mean_live(e^-S) / (Z + X mean_live(e^-S)); record; stop rule; live term.
__global__ void __launch_bounds__(1024)
ns_finish_kernel(NsArgs a, StepRecord* rec, int n_walk, HostPoll* hp) {
  pdl_enter();
  __shared__ double scratch[33];
  __shared__ float smin_s[33];
  Ctrl* ctrl = a.ctrl;
  if (ctrl->done) return;
  float m = INFINITY;
  for (int i = threadIdx.x; i < a.n; i += blockDim.x) m = fminf(m, a.S[i]);
  m = warp_min(m);
  if ((threadIdx.x & 31) == 0) smin_s[threadIdx.x >> 5] = m;
  __syncthreads();
  if (threadIdx.x < 32) {
    float v = threadIdx.x < (blockDim.x >> 5) ? smin_s[threadIdx.x] : INFINITY;
    v = warp_min(v);
    if (threadIdx.x == 0) smin_s[32] = v;
  }
  __syncthreads();
  const double smin = (double)smin_s[32];
  double acc = 0.0;
  for (int i = threadIdx.x; i < a.n; i += blockDim.x) acc += exp(-((double)a.S[i] - smin));
  acc = block_sum(acc, scratch);
  if (threadIdx.x == 0) {
    double log_live = ctrl->logX + (-smin + log(acc)) - log((double)a.n);
    double rem = exp(log_live - logaddexp_d(ctrl->logZ, log_live));
    int it = ctrl->temp_index;
    int fin = rem < a.stop_frac;
    if (it < a.max_iters) {
      StepRecord r;
      r.beta = ctrl->logX; r.delta = ctrl->S_star; r.ess_frac = rem; r.dlogZ = log_live;
      r.logZ = ctrl->logZ;
      r.accept_rate = (double)ctrl->n_accept / ((double)n_walk * (double)a.k_del);
      r.n_unique = 0; r.chol_status = ctrl->chol_status; r.index = it; r.done = fin;
      rec[it] = r;
    }
    ctrl->remaining = rem;
    ctrl->temp_index = it + 1;
    ctrl->n_accept = 0u;
    if (!isfinite(rem)) ctrl->nan_flag = 1;
    if (fin) {
      ctrl->logZ = logaddexp_d(ctrl->logZ, log_live);
      ctrl->done = 1;
    } else if (it + 1 >= a.max_iters) {
      ctrl->done = 2;   // dead-point log is full: stop without the live term
    }
    if (hp) {           // report to the host's run loop (see HostPoll)
      volatile HostPoll* v = hp;
      v->done = ctrl->done; v->nan_flag = ctrl->nan_flag; v->chol_status = ctrl->chol_status;
      __threadfence_system();
      v->seq = it + 1;
    }
  }
}

void launch_ns_finish(const NsArgs& a, StepRecord* rec, int n_walk, HostPoll* hp, cudaStream_t st) {
  ++g_launches; launch_pdl(ns_finish_kernel, 1, 1024, 0, st, a, rec, n_walk, hp);
}

// Posterior sample for `observables`: dead points (weight w_j e^{-S_j}) followed by the live
// points (weight X/n e^{-S_i}).  M_all[n_dead..] must already hold the live magnetisations.
__global__ void ns_obs_inputs_kernel(NsArgs a, int n_dead, float* M_all, float* S_all,
                                     double* logw_all) {
  int i = blockIdx.x * blockDim.x + threadIdx.x;
  if (i < n_dead) {
    M_all[i] = a.dead_M[i];
    S_all[i] = a.dead_S[i];
    logw_all[i] = a.dead_logw[i] - (double)a.dead_S[i];
  } else if (i < n_dead + a.n) {
    int l = i - n_dead;
    S_all[i] = a.S[l];
    logw_all[i] = a.ctrl->logX - log((double)a.n) - (double)a.S[l];
  }
}

void launch_ns_obs_inputs(const NsArgs& a, int n_dead, float* M_all, float* S_all,
                          double* logw_all, cudaStream_t st) {
  int tot = n_dead + a.n;
  ++g_launches; ns_obs_inputs_kernel<<<(tot + 255) / 256, 256, 0, st>>>(a, n_dead, M_all, S_all, logw_all);
}

}  // namespace phi4
