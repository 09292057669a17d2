// common.cuh -- shared declarations of the sm_100a kernels behind include/phi4smc.h.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

namespace phi4 {

// Number of kernels this library has launched (diagnostic; bench.py reports it as gpu_launches).
extern unsigned long long g_launches;

// Philox stream tags (reading R1).
enum : uint32_t {
  TAG_INIT = 0, TAG_PROP = 1, TAG_ACC = 2, TAG_RESAMPLE = 3,
  TAG_NS_START = 4, TAG_NS_PROP = 5, TAG_NS_ACC = 6, TAG_NS_SLICE = 7, TAG_Z2 = 8
};
enum : int { MODE_SMC = 0, MODE_NS = 1, MODE_IRMH = 2 };

// Device-resident control block: everything a temperature / NS iteration decides lives here so
// that a step can be enqueued without a host round trip.
struct Ctrl {
  double beta;        // current inverse temperature
  double delta;       // last increment
  double ess_frac;    // ESS/N at delta
  double dlogZ;
  double logZ;        // SMC: running sum; NS: log evidence from dead points (-inf at start)
  double logX;        // NS: log prior volume
  double S_star;      // NS: current threshold
  double remaining;   // NS: remaining evidence fraction
  float S_min;        // min S_E of the population at the last reweight
  int done;           // beta == 1 (SMC) / stop rule fired (NS)
  int temp_index;     // transitions / iterations completed
  int chol_fail;      // bit 0: plain attempt hit a pivot <= 0; bit 1: the jittered retry did too
  float trace;        // tr(Sigma) of the last covariance (jitter scale, reading A4)
  int chol_status;    // 0 plain, 1 jitter used, -1 failed
  int nan_flag;       // non-finite weight sum or action seen
  unsigned int n_accept;  // acceptances of the current mutation batch
  unsigned int n_unique;  // distinct ancestors of the last resampling
  unsigned long long q_total;  // T of reading R5
  unsigned long long mut_steps;  // SMC: mutation steps of the transitions completed since init / reset / restore
  unsigned int cta_done;  // CTAs of the fused mutation kernel that have finished (the last one closes the step)
};

// One record per temperature / iteration, written by the device at the end of each step.
struct StepRecord {
  double beta, delta, ess_frac, dlogZ, logZ, accept_rate;   // NS: logX, logZ, S_star, acc, rem
  int n_unique, chol_status, index, done;
};

// What the host needs to see of a finished temperature, written by the device straight into
// pinned host memory (seq last, after a system-wide fence): the run loop polls it without a
// copy in the stream, so the kernels of consecutive temperatures stay chained.
struct HostPoll { int seq, done, nan_flag, chol_status; };

// End of a temperature (one thread): record it, advance the index, latch done at beta == 1.
__device__ __forceinline__ void finish_step_device(Ctrl* ctrl, StepRecord* rec, int max_rec, int k, int N,
                                                   HostPoll* hp) {
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
  if (hp) {
    volatile HostPoll* v = hp;
    v->done = ctrl->done; v->nan_flag = ctrl->nan_flag; v->chol_status = ctrl->chol_status;
    __threadfence_system();
    v->seq = t + 1;
  }
}

// kappa: coefficient of the kinetic term (1 = Eq. 1; Eq. 2 scales it, reading A18).
// With kappa = 1 every kernel computes bit-for-bit what it computed before the field existed.
struct Model {
  int L, V;
  float m0sq, lam, kappa;
};

__host__ __device__ inline int round_up(int a, int b) { return (a + b - 1) / b * b; }

__device__ __forceinline__ float warp_sum(float v) {
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
  return v;
}
__device__ __forceinline__ double warp_sum(double v) {
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
  return v;
}
__device__ __forceinline__ float warp_min(float v) {
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) v = fminf(v, __shfl_xor_sync(0xffffffffu, v, o));
  return v;
}

// Block-wide sum of doubles; result valid in every thread.  scratch: >= 33 doubles of smem.
__device__ inline double block_sum(double v, double* scratch) {
  int lane = threadIdx.x & 31, w = threadIdx.x >> 5, nw = (blockDim.x + 31) >> 5;
  v = warp_sum(v);
  __syncthreads();
  if (lane == 0) scratch[w] = v;
  __syncthreads();
  if (w == 0) {
    double t = lane < nw ? scratch[lane] : 0.0;
    t = warp_sum(t);
    if (lane == 0) scratch[32] = t;
  }
  __syncthreads();
  return scratch[32];
}

// Programmatic dependent launch: a kernel launched through launch_pdl may be scheduled while its
// predecessor in the stream is still running; pdl_enter() -- the first statement of every such
// kernel -- lets the successor be scheduled in turn and then blocks until the predecessor has
// completed and its writes are visible (a grid's CTAs are only scheduled once every CTA of its
// predecessor has started, so waiting grids cannot starve the grids they wait for).  Stream order is unchanged; only the launch latency between
// the short dependent kernels of one temperature overlaps.  Launched normally, pdl_enter() is a
// no-op.  PHI4_NO_PDL=1 in the environment turns the attribute off.
__device__ __forceinline__ void pdl_trigger() {
  asm volatile("griddepcontrol.launch_dependents;" ::: "memory");
}
__device__ __forceinline__ void pdl_wait() { asm volatile("griddepcontrol.wait;" ::: "memory"); }
__device__ __forceinline__ void pdl_enter() {
  pdl_trigger();
  pdl_wait();
}

bool pdl_enabled();

template <typename... KArgs, typename... Args>
inline cudaError_t launch_pdl(void (*kernel)(KArgs...), dim3 grid, dim3 block, size_t smem,
                              cudaStream_t st, Args&&... args) {
  cudaLaunchConfig_t cfg = {};
  cfg.gridDim = grid; cfg.blockDim = block; cfg.dynamicSmemBytes = smem; cfg.stream = st;
  cudaLaunchAttribute at[1];
  at[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
  at[0].val.programmaticStreamSerializationAllowed = 1;
  cfg.attrs = at;
  cfg.numAttrs = pdl_enabled() ? 1 : 0;
  return cudaLaunchKernelEx(&cfg, kernel, KArgs(args)...);
}

}  // namespace phi4
