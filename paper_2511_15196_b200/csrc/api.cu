// api.cu -- the C ABI of include/phi4smc.h: handle, workspace carve-up, step sequencing.
// No torch types, no device allocation: all device state lives in the caller's workspace.
#include <chrono>
#include <math.h>
#include <stdio.h>
#include <stdlib.h>
#include <string.h>

#include <new>

#include "../../include/phi4smc.h"
#include "kernels.cuh"

#define PHI4_API extern "C" __attribute__((visibility("default")))

using namespace phi4;

namespace phi4 { unsigned long long g_launches = 0; }

namespace {
constexpr int KIND_SMC = 0, KIND_NS = 1;
constexpr int MAX_RECORDS = 4096;       // per-temperature records kept on the device (SMC)
constexpr size_t ALIGN = 256;

struct Carver {                         // bump allocator over the caller's workspace
  char* base;
  size_t off;
  template <typename T>
  T* take(size_t count) {
    off = (off + ALIGN - 1) / ALIGN * ALIGN;
    T* p = base ? reinterpret_cast<T*>(base + off) : nullptr;
    off += count * sizeof(T);
    return p;
  }
};
}  // namespace

struct phi4smc {
  int kind;
  Model md;
  int N, ld;                 // particles (n_live for NS) and padded stride
  uint64_t seed;
  smc_params prm;
  ns_params nsp;
  float s;                   // step scale actually used
  cudaStream_t st;
  // device state (inside the workspace)
  float* phi[2]; float* S[2]; float* U0[2];
  int cur;
  float *phip, *Z, *Z2, *w, *W2, *mu, *Sigma, *Lc, *Lsplit, *partial, *M, *margins;
  unsigned long long* C;
  int32_t* anc;
  uint8_t* acc_flags;
  Ctrl* ctrl;
  StepRecord* rec;
  int max_rec;
  double* obs_out;
  // nested sampling
  int k_del, n_walk, max_iters, ldw;
  double stop_frac;
  float *wphi, *wS, *wU, *dead_S, *dead_M, *M_all, *S_all;
  double *dead_logw, *logw_all, *hsum;
  int32_t *dead, *surv, *start, *gflag;
  unsigned long long* gkeys;
  // host side
  uint64_t step_counter;     // mutation steps enqueued so far (next step uses counter + 1)
  uint64_t step_base;        // steps not counted by the device: set_state / restore base + hook steps
  uint32_t iters_enqueued;   // NS iterations enqueued
  int64_t iter_base;         // NS: iters_enqueued - ctrl->temp_index after a set_state
  int known_done;
  Ctrl* h_ctrl;              // pinned staging
  HostPoll* h_hp;            // pinned, written by the device at the end of every SMC temperature
  // side stream (fork / join by events on the caller's stream; host resources only): nested
  // sampling runs the dead-point selection beside the covariance chain
  cudaStream_t side;
  cudaEvent_t fork_ev, join_ev;
  StepRecord* h_rec;         // pinned staging (one record)
  double* h_obs;             // pinned staging (85 doubles)
  char err[256];
};

#define CU(call)                                                                     \
  do {                                                                               \
    cudaError_t e_ = (call);                                                         \
    if (e_ != cudaSuccess) {                                                         \
      snprintf(h->err, sizeof(h->err), "%s: %s", #call, cudaGetErrorString(e_));     \
      return PHI4_ECUDA;                                                             \
    }                                                                                \
  } while (0)

static int carve_smc(phi4smc* h, char* base, size_t* total) {
  const int V = h->md.V, ld = h->ld, N = h->N;
  Carver c{base, 0};
  const size_t field = (size_t)V * ld;
  for (int b = 0; b < 2; ++b) {
    h->phi[b] = c.take<float>(field);
    h->S[b] = c.take<float>(ld);
    h->U0[b] = c.take<float>(ld);
  }
  h->phip = c.take<float>(field);
  {
    // normal scratch: [V][ld] (generic path), or the split normals / centred-split particles of
    // the tcgen05 paths, whichever is larger
    size_t zf = field;
    if (propose_tc_supported(V) && propose_tc_zsplit_floats(V, ld) > zf) zf = propose_tc_zsplit_floats(V, ld);
    if (syrk_tc_supported(V, ld) && syrk_tc_scratch_floats(V, ld) > zf) zf = syrk_tc_scratch_floats(V, ld);
    h->Z = c.take<float>(zf);
    // second buffer of split normals: step t+1 is drawn while step t multiplies (launch_mutate_generic)
    h->Z2 = propose_tc_supported(V) ? c.take<float>(propose_tc_zsplit_floats(V, ld)) : nullptr;
  }
  h->w = c.take<float>(ld);
  h->W2 = c.take<float>(ld);                               // IRMH: |Lc^-1 (phi - mu)|^2
  h->M = c.take<float>(ld);
  h->C = c.take<unsigned long long>(ld + 256);            // + block sums of the two-launch scan
  h->anc = c.take<int32_t>(ld);
  h->mu = c.take<float>(V);
  h->Sigma = c.take<float>((size_t)V * V);
  h->Lc = c.take<float>((size_t)V * V);
  h->partial = c.take<float>(cov_partial_floats(V, N));
  h->Lsplit = c.take<float>(mutate_tc_supported(V) ? mutate_tc_lsplit_floats(V) : (propose_tc_supported(V) ? propose_tc_lsplit_floats(V) : 4));
  h->acc_flags = c.take<uint8_t>((size_t)PHI4_MAX_HOOK_STEPS * N);
  h->margins = c.take<float>((size_t)PHI4_MAX_HOOK_STEPS * N);
  h->ctrl = c.take<Ctrl>(1);
  h->rec = c.take<StepRecord>(h->max_rec);
  h->obs_out = c.take<double>(5 + PHI4_HIST_BINS);
  *total = c.off + ALIGN;
  return 0;
}

static int carve_ns(phi4smc* h, char* base, size_t* total) {
  const int V = h->md.V, ld = h->ld, N = h->N, kd = h->k_del, ldw = h->ldw;
  Carver c{base, 0};
  h->phi[0] = c.take<float>((size_t)V * ld);
  h->S[0] = c.take<float>(ld);
  h->U0[0] = c.take<float>(ld);
  h->phi[1] = nullptr; h->S[1] = nullptr; h->U0[1] = nullptr;
  h->wphi = c.take<float>((size_t)V * ldw);
  h->wS = c.take<float>(ldw);
  h->wU = c.take<float>(ldw);
  h->phip = c.take<float>((size_t)V * ldw);
  h->Z = c.take<float>(propose_tc_supported(V) ? propose_tc_zsplit_floats(V, ldw) : (size_t)V * ldw);
  h->Z2 = propose_tc_supported(V) ? c.take<float>(propose_tc_zsplit_floats(V, ldw)) : nullptr;
  h->mu = c.take<float>(V);
  h->Sigma = c.take<float>((size_t)V * V);
  h->Lc = c.take<float>((size_t)V * V);
  h->partial = c.take<float>(cov_partial_floats(V, N));
  h->Lsplit = c.take<float>(mutate_tc_supported(V) ? mutate_tc_lsplit_floats(V) : (propose_tc_supported(V) ? propose_tc_lsplit_floats(V) : 4));
  h->dead = c.take<int32_t>(kd);
  h->surv = c.take<int32_t>(N);
  h->start = c.take<int32_t>(kd);
  h->gkeys = c.take<unsigned long long>(ns_sort_scratch_keys(N));
  h->gflag = c.take<int32_t>(ns_sort_scratch_keys(N) ? N : 0);
  const size_t nlog = (size_t)h->max_iters * kd;
  h->dead_S = c.take<float>(nlog);
  h->dead_M = c.take<float>(nlog);
  h->dead_logw = c.take<double>(nlog);
  h->hsum = c.take<double>(2 * kd + 1);
  h->M_all = c.take<float>(nlog + N);
  h->S_all = c.take<float>(nlog + N);
  h->logw_all = c.take<double>(nlog + N);
  h->acc_flags = c.take<uint8_t>((size_t)PHI4_MAX_HOOK_STEPS * kd);
  h->margins = c.take<float>((size_t)PHI4_MAX_HOOK_STEPS * kd);
  h->ctrl = c.take<Ctrl>(1);
  h->rec = c.take<StepRecord>(h->max_rec);
  h->obs_out = c.take<double>(5 + PHI4_HIST_BINS);
  *total = c.off + ALIGN;
  return 0;
}

static phi4smc* new_handle(int kind, int L, float kappa, float m0sq, float lambda, int N,
                           uint64_t seed) {
  phi4smc* h = new (std::nothrow) phi4smc;
  if (!h) return nullptr;
  memset(h, 0, sizeof(*h));
  h->kind = kind;
  h->md.L = L; h->md.V = L * L; h->md.m0sq = m0sq; h->md.lam = lambda;
  h->md.kappa = kappa;
  h->N = N; h->ld = round_up(N, 128);
  h->seed = seed;
  h->prm.k_steps = 10; h->prm.ess_target = 0.5f; h->prm.step_scale = 0.f; h->prm.mutation_path = 0;
  h->prm.kernel = 0; h->prm.hmc_eps = 0.1f; h->prm.hmc_leapfrog = 20; h->prm.z2_flip = 0;
  h->nsp.inner = 0; h->nsp.slice_width = 1.0f; h->nsp.max_expand = 8; h->nsp.max_shrink = 32;
  h->s = 2.38f / sqrtf((float)h->md.V);
  return h;
}

PHI4_API const char* phi4_strerror(int code) {
  switch (code) {
    case PHI4_OK: return "ok";
    case PHI4_EINVAL: return "invalid argument";
    case PHI4_ENOMEM: return "out of host memory";
    case PHI4_ENOTPD: return "particle covariance not positive definite";
    case PHI4_ENAN: return "non-finite action or weight";
    case PHI4_ECUDA: return "CUDA error or no device";
    case PHI4_ETRUNC: return "nested sampling stopped by max_iters: log_Z lacks the live-point term";
    case PHI4_ETOOBIG: return "size exceeds the fixed capacity of a no-allocation entry point (N > PHI4_NOALLOC_MAX_N = 131072)";
    default: return "unknown error";
  }
}

PHI4_API uint64_t phi4_kernel_launches(void) { return g_launches; }

// a failed *_init has no handle to carry its message: kept here, read with a NULL handle
static char g_init_err[256] = "";
static int init_failed(phi4smc* h, int rc) {
  snprintf(g_init_err, sizeof(g_init_err), "%s", h->err);
  delete h;
  return rc;
}

PHI4_API const char* phi4_last_cuda_error(const phi4smc* h) { return h ? h->err : g_init_err; }

PHI4_API size_t smc_workspace_bytes(int L, int N) {
  if (L < 1 || N < 2 || L > PHI4_MAX_L) return 0;
  phi4smc tmp;
  memset(&tmp, 0, sizeof(tmp));
  tmp.md.L = L; tmp.md.V = L * L; tmp.N = N; tmp.ld = round_up(N, 128); tmp.max_rec = MAX_RECORDS;
  size_t total = 0;
  carve_smc(&tmp, nullptr, &total);
  return total;
}

PHI4_API size_t ns_workspace_bytes(int L, int n_live, int k_delete, int max_iters) {
  if (L < 1 || L > PHI4_MAX_L || n_live < 2 || n_live > PHI4_NS_MAX_LIVE || k_delete < 1 ||
      k_delete >= n_live || max_iters < 1)
    return 0;
  phi4smc tmp;
  memset(&tmp, 0, sizeof(tmp));
  tmp.md.L = L; tmp.md.V = L * L; tmp.N = n_live; tmp.ld = round_up(n_live, 128);
  tmp.k_del = k_delete; tmp.ldw = round_up(k_delete, 128); tmp.max_iters = max_iters;
  tmp.max_rec = max_iters;
  size_t total = 0;
  carve_ns(&tmp, nullptr, &total);
  return total;
}

static int host_staging(phi4smc* h) {
  CU(cudaMallocHost((void**)&h->h_ctrl, sizeof(Ctrl)));
  CU(cudaMallocHost((void**)&h->h_hp, sizeof(HostPoll)));
  memset(h->h_hp, 0, sizeof(HostPoll));
  {
    CU(cudaStreamCreateWithFlags(&h->side, cudaStreamNonBlocking));
    CU(cudaEventCreateWithFlags(&h->fork_ev, cudaEventDisableTiming));
    CU(cudaEventCreateWithFlags(&h->join_ev, cudaEventDisableTiming));
  }
  CU(cudaMallocHost((void**)&h->h_rec, sizeof(StepRecord)));
  CU(cudaMallocHost((void**)&h->h_obs, sizeof(double) * (5 + PHI4_HIST_BINS)));
  return PHI4_OK;
}

static int have_device(phi4smc* h) {
  int n = 0;
  cudaError_t e = cudaGetDeviceCount(&n);
  if (e != cudaSuccess || n < 1) {
    snprintf(h->err, sizeof(h->err), "no CUDA device: %s", cudaGetErrorString(e));
    return PHI4_ECUDA;
  }
  return PHI4_OK;
}

// Pull the control block to the host (synchronises) and map device flags to error codes.
static int sync_ctrl(phi4smc* h) {
  CU(cudaMemcpyAsync(h->h_ctrl, h->ctrl, sizeof(Ctrl), cudaMemcpyDeviceToHost, h->st));
  CU(cudaStreamSynchronize(h->st));
  CU(cudaGetLastError());
  if (h->h_ctrl->done) h->known_done = 1;
  // the stream is idle: what the device counted is what ran (steps enqueued past the end of the
  // run were no-ops and are not in these counts)
  if (h->kind == KIND_SMC) h->step_counter = h->step_base + h->h_ctrl->mut_steps;
  else h->iters_enqueued = (uint32_t)(h->iter_base + (int64_t)h->h_ctrl->temp_index);
  if (h->h_ctrl->nan_flag) return PHI4_ENAN;
  if (h->h_ctrl->chol_status < 0) return PHI4_ENOTPD;
  return PHI4_OK;
}

static int push_ctrl(phi4smc* h) {
  CU(cudaMemcpyAsync(h->ctrl, h->h_ctrl, sizeof(Ctrl), cudaMemcpyHostToDevice, h->st));
  CU(cudaStreamSynchronize(h->st));
  return PHI4_OK;
}

// ------------------------------------------------------------------------------ SMC ----------
static int smc_init_impl(phi4smc** out, int L, float kappa, float m0sq, float lambda, int N,
                         uint64_t seed, void* d_workspace, size_t workspace_bytes,
                         void* cuda_stream) {
  if (!out) return PHI4_EINVAL;
  *out = nullptr;
  if (!isfinite(kappa) || !isfinite(m0sq) || !isfinite(lambda)) return PHI4_EINVAL;
  size_t need = smc_workspace_bytes(L, N);
  if (need == 0 || !d_workspace || workspace_bytes < need ||
      (reinterpret_cast<uintptr_t>(d_workspace) % ALIGN) != 0)
    return PHI4_EINVAL;
  phi4smc* h = new_handle(KIND_SMC, L, kappa, m0sq, lambda, N, seed);
  if (!h) return PHI4_ENOMEM;
  h->st = reinterpret_cast<cudaStream_t>(cuda_stream);
  h->max_rec = MAX_RECORDS;
  int rc = have_device(h);
  if (rc == PHI4_OK) rc = host_staging(h);
  if (rc != PHI4_OK) return init_failed(h, rc);
  size_t total;
  carve_smc(h, static_cast<char*>(d_workspace), &total);
  *out = h;
  CU(cudaMemsetAsync(d_workspace, 0, need, h->st));
  launch_init_particles(h->phi[0], N, h->ld, h->md.V, seed, h->st);
  launch_action(h->phi[0], N, h->ld, h->md, h->S[0], h->U0[0], h->ctrl, h->st);
  launch_set_identity(h->Lc, h->md.V, h->st);
  CU(cudaGetLastError());
  return PHI4_OK;
}

PHI4_API int smc_init(phi4smc** out, int L, float m0sq, float lambda, int N, uint64_t seed,
                        void* d_workspace, size_t workspace_bytes, void* cuda_stream) {
  return smc_init_impl(out, L, 1.0f, m0sq, lambda, N, seed, d_workspace, workspace_bytes,
                       cuda_stream);
}

// Eq. 2 -> Eq. 1 coefficients by Eq. 4 (reading A18): kinetic kappa,
// m0^2 = 2 (1 - 2 lambda), quartic lambda; the constant V lambda is dropped as in Eq. 5.
PHI4_API int smc_init_kl(phi4smc** out, int L, float kappa, float lambda, int N, uint64_t seed,
                           void* d_workspace, size_t workspace_bytes, void* cuda_stream) {
  if (!(kappa >= 0.f) || !(lambda >= 0.f)) { if (out) *out = nullptr; return PHI4_EINVAL; }
  return smc_init_impl(out, L, kappa, 2.0f * (1.0f - 2.0f * lambda), lambda, N, seed, d_workspace,
                       workspace_bytes, cuda_stream);
}

PHI4_API int smc_reset(phi4smc* h, uint64_t seed) {
  if (!h) return PHI4_EINVAL;
  h->seed = seed;
  h->cur = 0;
  h->step_counter = 0;
  h->step_base = 0;
  h->iters_enqueued = 0;
  h->iter_base = 0;
  h->known_done = 0;
  // h_ctrl is pinned staging that an earlier async copy may still be reading: use a memset for
  // the zero state and a tiny kernel-free patch for the NS evidence (-inf) via a second copy.
  CU(cudaMemsetAsync(h->ctrl, 0, sizeof(Ctrl), h->st));
  if (h->kind == KIND_NS) {
    static const double neg_inf = -INFINITY;
    CU(cudaMemcpyAsync(&h->ctrl->logZ, &neg_inf, sizeof(double), cudaMemcpyHostToDevice, h->st));
  }
  launch_init_particles(h->phi[0], h->N, h->ld, h->md.V, seed, h->st);
  launch_action(h->phi[0], h->N, h->ld, h->md, h->S[0], h->U0[0], h->ctrl, h->st);
  launch_set_identity(h->Lc, h->md.V, h->st);
  CU(cudaGetLastError());
  return PHI4_OK;
}

PHI4_API int smc_destroy(phi4smc* h) {
  if (!h) return PHI4_OK;
  cudaStreamSynchronize(h->st);
  if (h->h_ctrl) cudaFreeHost(h->h_ctrl);
  if (h->h_hp) cudaFreeHost(h->h_hp);
  if (h->side) { cudaStreamSynchronize(h->side); cudaStreamDestroy(h->side); }
  if (h->fork_ev) cudaEventDestroy(h->fork_ev);
  if (h->join_ev) cudaEventDestroy(h->join_ev);
  if (h->h_rec) cudaFreeHost(h->h_rec);
  if (h->h_obs) cudaFreeHost(h->h_obs);
  delete h;
  return PHI4_OK;
}

PHI4_API int smc_set_params(phi4smc* h, const smc_params* p) {
  if (!h || !p) return PHI4_EINVAL;
  if (p->k_steps < 1 || !(p->ess_target > 0.f && p->ess_target < 1.f) || p->step_scale < 0.f ||
      p->mutation_path < 0 || p->mutation_path > 3)
    return PHI4_EINVAL;
  if (p->mutation_path == 2 && !mutate_tc_supported(h->md.V) && !propose_tc_supported(h->md.V))
    return PHI4_EINVAL;
  if (p->mutation_path == 3 && !propose_tc_supported(h->md.V)) return PHI4_EINVAL;
  if (p->kernel < 0 || p->kernel > 2 || p->z2_flip < 0 || p->z2_flip > 1) return PHI4_EINVAL;
  if (p->kernel == 2 && (h->kind != KIND_SMC || !irmh_supported(h->md.V))) return PHI4_EINVAL;
  if (p->kernel == 1 && (h->kind != KIND_SMC || !(p->hmc_eps > 0.f) || p->hmc_leapfrog < 1))
    return PHI4_EINVAL;
  h->prm = *p;
  h->s = p->step_scale > 0.f ? p->step_scale : 2.38f / sqrtf((float)h->md.V);
  return PHI4_OK;
}

static MutateArgs smc_mutate_args(phi4smc* h, int k, uint8_t* acc, float* mar, int respect_done) {
  MutateArgs a;
  a.phi = h->phi[h->cur]; a.phip = h->phip; a.Z = h->Z;
  a.Z2 = h->Z2;
  a.S = h->S[h->cur]; a.U0 = h->U0[h->cur]; a.Lc = h->Lc; a.ctrl = h->ctrl;
  a.acc_out = acc; a.margin_out = mar;
  a.N = h->N; a.ld = h->ld; a.md = h->md; a.s = h->s; a.mode = MODE_SMC; a.seed = h->seed;
  a.tag_prop = TAG_PROP; a.tag_acc = TAG_ACC;
  a.t0 = (uint32_t)(h->step_counter + 1); a.k = k; a.respect_done = respect_done;
  a.tc_f16 = h->prm.mutation_path != 3;
  return a;
}

// mutation_path 0: the fused tcgen05 kernel whenever it supports this V, else the generic path
static bool use_tc_path(const phi4smc* h) {
  return h->prm.mutation_path != 1 && mutate_tc_supported(h->md.V);
}

// large V: tcgen05 proposal GEMM + the generic accept step
static bool use_tc_propose(const phi4smc* h) {
  return h->prm.mutation_path != 1 && propose_tc_supported(h->md.V);
}

static void enqueue_mutation(phi4smc* h, const MutateArgs& a) {
  if (h->prm.kernel == 1 && a.mode == MODE_SMC && !hmc_supported(a.md.V)) {
    // positions double-buffered in phip and the second half of the normal scratch (2 V ld floats
    // whenever the tcgen05 proposal exists, i.e. for every V this path serves), momenta in its first
    launch_hmc_generic(a.phi, a.S, a.U0, h->Sigma, a.phip, a.Z + (size_t)a.md.V * a.ld, a.Z, h->W2, a.N, a.ld, a.md, h->prm.hmc_eps,
                       h->prm.hmc_leapfrog, a.seed, a.t0, a.k, a.ctrl, a.acc_out, a.margin_out,
                       a.respect_done, h->st);
    return;
  }
  if (h->prm.kernel == 1 && a.mode == MODE_SMC) {
    launch_hmc(a.phi, a.S, a.U0, h->Sigma, a.N, a.ld, a.md, h->prm.hmc_eps, h->prm.hmc_leapfrog,
               a.seed, a.t0, a.k, a.ctrl, a.acc_out, a.margin_out, a.respect_done, h->st);
    return;
  }
  if (h->prm.kernel == 2 && a.mode == MODE_SMC) {
    launch_mutate_irmh(a, h->mu, h->W2,
                       (h->prm.mutation_path != 1 && mutate_tc_supported(a.md.V, true)) ? h->Lsplit : nullptr, h->st);
    return;
  }
  if (use_tc_path(h)) launch_mutate_tc(a, h->Lsplit, h->st);
  else launch_mutate_generic(a, use_tc_propose(h) ? h->Lsplit : nullptr, h->st);
}

static CovCholArgs cov_args(phi4smc* h, int respect_done) {
  CovCholArgs c;
  c.phi = h->phi[h->cur]; c.N = h->N; c.ld = h->ld; c.V = h->md.V;
  c.mu = h->mu; c.Sigma = h->Sigma; c.Lc = h->Lc; c.partial = h->partial; c.ctrl = h->ctrl;
  // the split-normal scratch of the large-V proposal doubles as the centred-split scratch
  c.tc_scratch = (h->prm.mutation_path != 1 && propose_tc_supported(h->md.V) && h->kind == KIND_SMC) ? h->Z : nullptr;
  c.tc_small = h->prm.mutation_path != 1;
  c.tc_f16 = h->prm.mutation_path != 3;
  c.respect_done = respect_done;
  return c;
}

static void enqueue_resample(phi4smc* h, bool scanned = false) {
  if (!scanned) launch_quantise_scan(h->w, h->N, h->C, h->ctrl, h->st);
  // the accept-flag scratch of the hooks doubles as the per-slot Z2 flip bytes
  launch_ancestors(h->C, h->N, h->seed, h->anc, h->acc_flags, h->prm.z2_flip, h->ctrl, h->st);
  const int o = h->cur ^ 1;
  launch_gather(h->phi[h->cur], h->phi[o], h->S[h->cur], h->S[o], h->U0[h->cur], h->U0[o], h->anc,
                h->prm.z2_flip ? h->acc_flags : nullptr,
                h->N, h->ld, h->md.V, h->ctrl, h->st);
  h->cur = o;
}

static void enqueue_smc_step(phi4smc* h) {
  const bool scanned = launch_next_delta_reweight(h->S[h->cur], h->N, h->prm.ess_target, -1.0, h->w,
                                                  h->C, h->ctrl, h->st);
  enqueue_resample(h, scanned);
  launch_cov_chol(cov_args(h, 1), h->st);
  MutateArgs a = smc_mutate_args(h, h->prm.k_steps, nullptr, nullptr, 1);
  // the fused tcgen05 mutation closes the temperature itself (its last CTA); the other mutation
  // paths are several launches, so the step is closed by a kernel of its own
  const bool fused_finish = (h->prm.kernel == 0 && use_tc_path(h)) ||
                            (h->prm.kernel == 2 && h->prm.mutation_path != 1 && mutate_tc_supported(h->md.V, true));
  if (fused_finish) { a.finish_rec = h->rec; a.finish_max_rec = h->max_rec; a.finish_poll = h->h_hp; }
  enqueue_mutation(h, a);
  h->step_counter += (uint64_t)h->prm.k_steps;
  if (!fused_finish) launch_finish_step(h->ctrl, h->rec, h->max_rec, h->prm.k_steps, h->N, h->h_hp, h->st);
}

static void fill_info(const StepRecord& r, smc_step_info* info) {
  info->beta = r.beta; info->delta = r.delta; info->ess_frac = r.ess_frac; info->dlogZ = r.dlogZ;
  info->logZ = r.logZ; info->accept_rate = r.accept_rate; info->n_unique = r.n_unique;
  info->chol_status = r.chol_status; info->temp_index = r.index; info->done = r.done;
}

static int fetch_record(phi4smc* h, int index, StepRecord* out) {
  if (index < 0 || index >= h->max_rec) return PHI4_EINVAL;
  CU(cudaMemcpyAsync(h->h_rec, h->rec + index, sizeof(StepRecord), cudaMemcpyDeviceToHost, h->st));
  CU(cudaStreamSynchronize(h->st));
  *out = *h->h_rec;
  return PHI4_OK;
}

PHI4_API int smc_step(phi4smc* h, smc_step_info* info) {
  if (!h || h->kind != KIND_SMC) return PHI4_EINVAL;
  if (!h->known_done) enqueue_smc_step(h);
  if (!info) {
    CU(cudaGetLastError());
    return PHI4_OK;
  }
  int rc = sync_ctrl(h);
  if (rc == PHI4_ECUDA) return rc;
  memset(info, 0, sizeof(*info));
  int last = h->h_ctrl->temp_index - 1;
  if (last >= 0 && last < h->max_rec) {
    StepRecord r;
    int rr = fetch_record(h, last, &r);
    if (rr != PHI4_OK) return rr;
    fill_info(r, info);
  } else if (last >= 0) {
    // the history is full: report the control block (accept_rate / n_unique are not kept there)
    const Ctrl& c = *h->h_ctrl;
    info->beta = c.beta; info->delta = c.delta; info->ess_frac = c.ess_frac; info->dlogZ = c.dlogZ;
    info->logZ = c.logZ; info->chol_status = c.chol_status; info->temp_index = last;
  }
  info->done = h->h_ctrl->done ? 1 : 0;
  return rc;
}

// Shared by smc_run / ns_run.  The device reports every finished step in pinned host memory
// (HostPoll, written by the kernel that closes the step): no copy or event sits in the stream
// between two steps, so their kernels stay chained.  One step is kept queued behind the one whose
// report the host is waiting for.  `start` = steps completed before this call.
constexpr int RUN_STALL_SECONDS = 120;
template <typename F>
static int run_polled(phi4smc* h, int max_steps, int start, F enqueue) {
  volatile HostPoll* hp = h->h_hp;
  hp->seq = start; hp->done = h->h_ctrl->done; hp->nan_flag = h->h_ctrl->nan_flag;
  hp->chol_status = h->h_ctrl->chol_status;
  if (h->h_ctrl->done) h->known_done = 1;
  int enq = 0;
  while (!h->known_done && enq < max_steps) {
    enqueue(h);
    ++enq;
    if (enq >= 2) {
      const int target = start + enq - 1;        // the step before the one just enqueued
      int seen = hp->seq;
      auto moved = std::chrono::steady_clock::now();
      for (unsigned spin = 1; hp->seq < target && !hp->done; ++spin) {
        if ((spin & 1023u) == 0) {               // a dead stream must not hang the host
          cudaError_t q = cudaStreamQuery(h->st);
          if (q == cudaSuccess) break;
          if (q != cudaErrorNotReady) {
            snprintf(h->err, sizeof(h->err), "run: %s", cudaGetErrorString(q));
            return PHI4_ECUDA;
          }
          // ... nor a stream that stopped making progress (no step takes anywhere near this long)
          const auto now = std::chrono::steady_clock::now();
          if (hp->seq != seen) { seen = hp->seq; moved = now; }
          else if (now - moved > std::chrono::seconds(RUN_STALL_SECONDS)) {
            snprintf(h->err, sizeof(h->err), "run: no step finished for %d s (device stalled at step %d)",
                     RUN_STALL_SECONDS, seen);
            return PHI4_ECUDA;
          }
        }
      }
      if (hp->done) h->known_done = 1;
      if (hp->nan_flag || hp->chol_status < 0) break;
    }
  }
  return sync_ctrl(h);
}

PHI4_API int smc_run(phi4smc* h, int max_temps, int* n_temps) {
  if (!h || h->kind != KIND_SMC || max_temps < 0) return PHI4_EINVAL;
  int rc = sync_ctrl(h);
  if (rc != PHI4_OK) return rc;
  const int start = h->h_ctrl->temp_index;
  rc = run_polled(h, max_temps, start, enqueue_smc_step);
  // (steps enqueued past beta = 1 were no-ops; sync_ctrl took the step counter from the device)
  const int made = h->h_ctrl->temp_index - start;
  if (n_temps) *n_temps = made;
  return rc;
}

PHI4_API int smc_get_history(phi4smc* h, smc_step_info* h_info, int cap, int* n) {
  if (!h || h->kind != KIND_SMC) return PHI4_EINVAL;
  int rc = sync_ctrl(h);
  if (rc == PHI4_ECUDA) return rc;
  int avail = h->h_ctrl->temp_index < h->max_rec ? h->h_ctrl->temp_index : h->max_rec;
  if (n) *n = avail;
  int m = avail < cap ? avail : cap;
  if (h_info && m > 0) {
    StepRecord* tmp = (StepRecord*)malloc(sizeof(StepRecord) * m);
    if (!tmp) return PHI4_ENOMEM;
    cudaError_t e = cudaMemcpy(tmp, h->rec, sizeof(StepRecord) * m, cudaMemcpyDeviceToHost);
    if (e != cudaSuccess) { free(tmp); snprintf(h->err, sizeof(h->err), "history: %s", cudaGetErrorString(e)); return PHI4_ECUDA; }
    for (int i = 0; i < m; ++i) fill_info(tmp[i], &h_info[i]);
    free(tmp);
  }
  return PHI4_OK;
}

PHI4_API int estimate_cov_chol(phi4smc* h) {
  if (!h) return PHI4_EINVAL;
  launch_cov_chol(cov_args(h, 0), h->st);
  CU(cudaGetLastError());
  return PHI4_OK;
}

static NsArgs ns_args(phi4smc* h);

PHI4_API int observables(phi4smc* h, phi4_observables* out) {
  if (!h || !out) return PHI4_EINVAL;
  const int V = h->md.V;
  if (h->kind == KIND_SMC) {
    launch_magnetisation(h->phi[h->cur], h->N, h->ld, V, h->M, h->st);
    launch_observables_reduce(h->M, h->S[h->cur], nullptr, h->N, V, h->obs_out, h->st);
  } else {
    int rc = sync_ctrl(h);
    if (rc == PHI4_ECUDA) return rc;
    int iters = h->h_ctrl->temp_index < h->max_iters ? h->h_ctrl->temp_index : h->max_iters;
    int n_dead = iters * h->k_del;
    launch_magnetisation(h->phi[0], h->N, h->ld, V, h->M_all + n_dead, h->st);
    launch_ns_obs_inputs(ns_args(h), n_dead, h->M_all, h->S_all, h->logw_all, h->st);
    launch_observables_reduce(h->M_all, h->S_all, h->logw_all, n_dead + h->N, V, h->obs_out, h->st);
  }
  CU(cudaMemcpyAsync(h->h_obs, h->obs_out, sizeof(double) * (5 + PHI4_HIST_BINS),
                     cudaMemcpyDeviceToHost, h->st));
  CU(cudaStreamSynchronize(h->st));
  CU(cudaGetLastError());
  out->absM = h->h_obs[0]; out->M2 = h->h_obs[1]; out->chi = h->h_obs[2];
  out->mean_SE = h->h_obs[3]; out->mode_balance = h->h_obs[4];
  for (int b = 0; b < PHI4_HIST_BINS; ++b) out->hist[b] = h->h_obs[5 + b];
  return PHI4_OK;
}

PHI4_API double log_Z(const phi4smc* hc) {
  phi4smc* h = const_cast<phi4smc*>(hc);
  if (!h) return NAN;
  if (sync_ctrl(h) == PHI4_ECUDA) return NAN;
  return h->h_ctrl->logZ;
}

// ------------------------------------------------------------------- nested sampling ---------
static NsArgs ns_args(phi4smc* h) {
  NsArgs a;
  a.phi = h->phi[0]; a.S = h->S[0]; a.U0 = h->U0[0];
  a.wphi = h->wphi; a.wS = h->wS; a.wU = h->wU;
  a.n = h->N; a.ld = h->ld; a.k_del = h->k_del; a.ldw = h->ldw; a.V = h->md.V;
  a.seed = h->seed; a.dead = h->dead; a.surv = h->surv; a.start = h->start;
  a.dead_S = h->dead_S; a.dead_M = h->dead_M; a.dead_logw = h->dead_logw;
  a.max_iters = h->max_iters; a.stop_frac = h->stop_frac; a.ctrl = h->ctrl; a.hsum = h->hsum;
  a.gkeys = h->gkeys; a.gflag = h->gflag;
  return a;
}

static int ns_init_impl(phi4smc** out, int L, float kappa, float m0sq, float lambda, int n_live,
                        int k_delete, int n_walk, uint64_t seed, double stop_frac, int max_iters,
                        void* d_workspace, size_t workspace_bytes, void* cuda_stream) {
  if (!out) return PHI4_EINVAL;
  *out = nullptr;
  if (n_live > PHI4_NS_MAX_LIVE || n_walk < 1 || !(stop_frac > 0.0)) return PHI4_EINVAL;
  if (!isfinite(kappa) || !isfinite(m0sq) || !isfinite(lambda)) return PHI4_EINVAL;
  size_t need = ns_workspace_bytes(L, n_live, k_delete, max_iters);
  if (need == 0 || !d_workspace || workspace_bytes < need ||
      (reinterpret_cast<uintptr_t>(d_workspace) % ALIGN) != 0)
    return PHI4_EINVAL;
  phi4smc* h = new_handle(KIND_NS, L, kappa, m0sq, lambda, n_live, seed);
  if (!h) return PHI4_ENOMEM;
  h->st = reinterpret_cast<cudaStream_t>(cuda_stream);
  h->k_del = k_delete; h->ldw = round_up(k_delete, 128); h->n_walk = n_walk;
  h->max_iters = max_iters; h->max_rec = max_iters; h->stop_frac = stop_frac;
  int rc = have_device(h);
  if (rc == PHI4_OK) rc = host_staging(h);
  if (rc != PHI4_OK) return init_failed(h, rc);
  size_t total;
  carve_ns(h, static_cast<char*>(d_workspace), &total);
  *out = h;
  CU(cudaMemsetAsync(d_workspace, 0, need, h->st));
  memset(h->h_ctrl, 0, sizeof(Ctrl));
  h->h_ctrl->logZ = -INFINITY;
  CU(cudaMemcpyAsync(h->ctrl, h->h_ctrl, sizeof(Ctrl), cudaMemcpyHostToDevice, h->st));
  launch_ns_hsum(h->hsum, n_live, k_delete, h->st);
  launch_init_particles(h->phi[0], n_live, h->ld, h->md.V, seed, h->st);
  launch_action(h->phi[0], n_live, h->ld, h->md, h->S[0], h->U0[0], h->ctrl, h->st);
  launch_set_identity(h->Lc, h->md.V, h->st);
  CU(cudaStreamSynchronize(h->st));
  CU(cudaGetLastError());
  return PHI4_OK;
}

PHI4_API int ns_init(phi4smc** out, int L, float m0sq, float lambda, int n_live, int k_delete,
                       int n_walk, uint64_t seed, double stop_frac, int max_iters,
                       void* d_workspace, size_t workspace_bytes, void* cuda_stream) {
  return ns_init_impl(out, L, 1.0f, m0sq, lambda, n_live, k_delete, n_walk, seed, stop_frac,
                      max_iters, d_workspace, workspace_bytes, cuda_stream);
}

PHI4_API int ns_init_kl(phi4smc** out, int L, float kappa, float lambda, int n_live, int k_delete,
                          int n_walk, uint64_t seed, double stop_frac, int max_iters,
                          void* d_workspace, size_t workspace_bytes, void* cuda_stream) {
  if (!(kappa >= 0.f) || !(lambda >= 0.f)) { if (out) *out = nullptr; return PHI4_EINVAL; }
  return ns_init_impl(out, L, kappa, 2.0f * (1.0f - 2.0f * lambda), lambda, n_live, k_delete,
                      n_walk, seed, stop_frac, max_iters, d_workspace, workspace_bytes,
                      cuda_stream);
}

static void enqueue_ns_step(phi4smc* h) {
  NsArgs a = ns_args(h);
  // N1 / N2 and the walker gather (S_E order, evidence, start points) read nothing the covariance
  // chain writes: they run beside it on the side stream (38 + 8 us hidden behind mean / syrk /
  // Cholesky, 50 us, at C2)
  cudaEventRecord(h->fork_ev, h->st);
  cudaStreamWaitEvent(h->side, h->fork_ev, 0);
  launch_ns_select_evidence(a, h->side);
  launch_ns_load_walkers(a, h->side);
  cudaEventRecord(h->join_ev, h->side);
  launch_cov_chol(cov_args(h, 1), h->st);
  cudaStreamWaitEvent(h->st, h->join_ev, 0);
  MutateArgs m;
  m.Z2 = h->Z2;
  m.phi = h->wphi; m.phip = h->phip; m.Z = h->Z; m.S = h->wS; m.U0 = h->wU; m.Lc = h->Lc;
  m.ctrl = h->ctrl; m.acc_out = nullptr; m.margin_out = nullptr;
  m.N = h->k_del; m.ld = h->ldw; m.md = h->md; m.s = h->s; m.mode = MODE_NS; m.seed = h->seed;
  m.tag_prop = TAG_NS_PROP; m.tag_acc = TAG_NS_ACC;
  m.t0 = h->iters_enqueued * (uint32_t)h->n_walk + 1u; m.k = h->n_walk; m.respect_done = 1;
  if (h->nsp.inner == 1) launch_ns_slice(m, h->nsp.slice_width, h->nsp.max_expand, h->nsp.max_shrink, h->st);
  else enqueue_mutation(h, m);
  launch_ns_store_walkers(a, h->st);
  launch_ns_finish(a, h->rec, h->n_walk, h->h_hp, h->st);
  h->iters_enqueued += 1;
}

PHI4_API int ns_set_params(phi4smc* h, const ns_params* p) {
  if (!h || !p || h->kind != KIND_NS) return PHI4_EINVAL;
  if (p->inner < 0 || p->inner > 1) return PHI4_EINVAL;
  if (p->inner == 1 && (!(p->slice_width > 0.f) || p->max_expand < 1 || p->max_expand > 64 ||
                        p->max_shrink < 1 || p->max_shrink > 256))
    return PHI4_EINVAL;
  h->nsp = *p;
  return PHI4_OK;
}

static void fill_ns_info(const StepRecord& r, ns_step_info* info) {
  info->logX = r.beta; info->S_star = r.delta; info->remaining_frac = r.ess_frac;
  info->logZ = r.logZ; info->accept_rate = r.accept_rate; info->chol_status = r.chol_status;
  info->iter_index = r.index; info->done = r.done;
}

PHI4_API int ns_step(phi4smc* h, ns_step_info* info) {
  if (!h || h->kind != KIND_NS) return PHI4_EINVAL;
  if (!h->known_done) enqueue_ns_step(h);
  if (!info) {
    CU(cudaGetLastError());
    return PHI4_OK;
  }
  int rc = sync_ctrl(h);
  if (rc == PHI4_ECUDA) return rc;
  memset(info, 0, sizeof(*info));
  int last = h->h_ctrl->temp_index - 1;
  if (last >= 0 && last < h->max_rec) {
    StepRecord r;
    int rr = fetch_record(h, last, &r);
    if (rr != PHI4_OK) return rr;
    fill_ns_info(r, info);
  }
  info->done = h->h_ctrl->done;                  // 0 running, 1 converged, 2 truncated
  return (rc == PHI4_OK && h->h_ctrl->done == 2) ? PHI4_ETRUNC : rc;
}

PHI4_API int ns_run(phi4smc* h, int max_iters, int* n_iters) {
  if (!h || h->kind != KIND_NS || max_iters < 0) return PHI4_EINVAL;
  int rc = sync_ctrl(h);
  if (rc != PHI4_OK) return rc;
  const int start = h->h_ctrl->temp_index;
  rc = run_polled(h, max_iters, start, enqueue_ns_step);
  const int made = h->h_ctrl->temp_index - start;
  if (n_iters) *n_iters = made;
  return (rc == PHI4_OK && h->h_ctrl->done == 2) ? PHI4_ETRUNC : rc;
}

PHI4_API int ns_get_dead(phi4smc* h, int32_t* h_last_dead_idx, float* h_dead_S, float* h_dead_M,
                           double* h_dead_logw, int cap, int* n_dead) {
  if (!h || h->kind != KIND_NS) return PHI4_EINVAL;
  int rc = sync_ctrl(h);
  if (rc == PHI4_ECUDA) return rc;
  int iters = h->h_ctrl->temp_index < h->max_iters ? h->h_ctrl->temp_index : h->max_iters;
  int nd = iters * h->k_del;
  if (n_dead) *n_dead = nd;
  int m = nd < cap ? nd : cap;
  if (h_last_dead_idx) CU(cudaMemcpy(h_last_dead_idx, h->dead, sizeof(int32_t) * h->k_del, cudaMemcpyDeviceToHost));
  if (h_dead_S && m > 0) CU(cudaMemcpy(h_dead_S, h->dead_S, sizeof(float) * m, cudaMemcpyDeviceToHost));
  if (h_dead_M && m > 0) CU(cudaMemcpy(h_dead_M, h->dead_M, sizeof(float) * m, cudaMemcpyDeviceToHost));
  if (h_dead_logw && m > 0) CU(cudaMemcpy(h_dead_logw, h->dead_logw, sizeof(double) * m, cudaMemcpyDeviceToHost));
  return PHI4_OK;
}

PHI4_API int ns_set_dead(phi4smc* h, const float* h_dead_S, const float* h_dead_M,
                           const double* h_dead_logw, int n_dead) {
  if (!h || h->kind != KIND_NS || n_dead < 0 || !h_dead_S || !h_dead_M || !h_dead_logw) return PHI4_EINVAL;
  if ((size_t)n_dead > (size_t)h->max_iters * h->k_del) return PHI4_EINVAL;
  CU(cudaStreamSynchronize(h->st));
  if (n_dead > 0) {
    CU(cudaMemcpy(h->dead_S, h_dead_S, sizeof(float) * n_dead, cudaMemcpyHostToDevice));
    CU(cudaMemcpy(h->dead_M, h_dead_M, sizeof(float) * n_dead, cudaMemcpyHostToDevice));
    CU(cudaMemcpy(h->dead_logw, h_dead_logw, sizeof(double) * n_dead, cudaMemcpyHostToDevice));
  }
  return PHI4_OK;
}

// ------------------------------------------------------------------------ hooks --------------
PHI4_API int smc_get_state(phi4smc* h, float* h_phi, float* h_SE, float* h_U0, double* beta,
                             uint64_t* step_counter) {
  if (!h) return PHI4_EINVAL;
  int rc = sync_ctrl(h);
  if (rc == PHI4_ECUDA) return rc;
  const int V = h->md.V, N = h->N, c = h->cur;
  if (h_phi)
    CU(cudaMemcpy2D(h_phi, sizeof(float) * N, h->phi[c], sizeof(float) * h->ld, sizeof(float) * N,
                    V, cudaMemcpyDeviceToHost));
  if (h_SE) CU(cudaMemcpy(h_SE, h->S[c], sizeof(float) * N, cudaMemcpyDeviceToHost));
  if (h_U0) CU(cudaMemcpy(h_U0, h->U0[c], sizeof(float) * N, cudaMemcpyDeviceToHost));
  if (beta) *beta = h->h_ctrl->beta;
  if (step_counter)
    *step_counter = h->kind == KIND_SMC ? h->step_counter
                                        : (uint64_t)h->iters_enqueued * (uint64_t)h->n_walk;
  return PHI4_OK;
}

PHI4_API int smc_set_state(phi4smc* h, const float* h_phi, double beta, uint64_t step_counter) {
  if (!h || !h_phi || !(beta >= 0.0 && beta <= 1.0)) return PHI4_EINVAL;
  int rc = sync_ctrl(h);
  if (rc == PHI4_ECUDA) return rc;
  const int V = h->md.V, N = h->N, c = h->cur;
  CU(cudaMemcpy2DAsync(h->phi[c], sizeof(float) * h->ld, h_phi, sizeof(float) * N,
                       sizeof(float) * N, V, cudaMemcpyHostToDevice, h->st));
  h->h_ctrl->beta = beta;
  h->h_ctrl->done = (h->kind == KIND_SMC && beta >= 1.0) ? 1 : 0;
  h->h_ctrl->nan_flag = 0;
  h->h_ctrl->mut_steps = 0;
  h->known_done = h->h_ctrl->done;
  rc = push_ctrl(h);
  if (rc != PHI4_OK) return rc;
  launch_action(h->phi[c], N, h->ld, h->md, h->S[c], h->U0[c], h->ctrl, h->st);
  if (h->kind == KIND_SMC) {
    h->step_counter = h->step_base = step_counter;
  } else {
    h->iters_enqueued = (uint32_t)(step_counter / (uint64_t)h->n_walk);
    h->iter_base = (int64_t)h->iters_enqueued - (int64_t)h->h_ctrl->temp_index;
  }
  CU(cudaStreamSynchronize(h->st));
  CU(cudaGetLastError());
  return PHI4_OK;
}

// Checkpoint / resume (bit for bit): the scalars of the control block that smc_get_state does not
// return, and a restore that also takes the cached S_E / U0 (recomputing them would differ from
// the incrementally updated values by fp32 rounding, and the weights are formed from them).
PHI4_API int smc_get_run_state(phi4smc* h, phi4_run_state* out) {
  if (!h || !out) return PHI4_EINVAL;
  int rc = sync_ctrl(h);
  if (rc == PHI4_ECUDA) return rc;
  const Ctrl& c = *h->h_ctrl;
  memset(out, 0, sizeof(*out));
  out->beta = c.beta; out->delta = c.delta; out->logZ = c.logZ; out->logX = c.logX;
  out->S_star = c.S_star; out->remaining_frac = c.remaining;
  out->index = c.temp_index; out->done = c.done;
  out->step_counter = h->kind == KIND_SMC ? h->step_counter
                                          : (uint64_t)h->iters_enqueued * (uint64_t)h->n_walk;
  return PHI4_OK;
}

PHI4_API int smc_restore(phi4smc* h, const float* h_phi, const float* h_SE, const float* h_U0,
                           const phi4_run_state* rs) {
  if (!h || !h_phi || !rs || rs->index < 0 || !(rs->beta >= 0.0 && rs->beta <= 1.0)) return PHI4_EINVAL;
  if ((h_SE == nullptr) != (h_U0 == nullptr)) return PHI4_EINVAL;
  int rc = sync_ctrl(h);
  if (rc == PHI4_ECUDA) return rc;
  const int V = h->md.V, N = h->N, c = h->cur;
  CU(cudaMemcpy2DAsync(h->phi[c], sizeof(float) * h->ld, h_phi, sizeof(float) * N,
                       sizeof(float) * N, V, cudaMemcpyHostToDevice, h->st));
  Ctrl z;
  memset(&z, 0, sizeof(z));
  z.beta = rs->beta; z.delta = rs->delta; z.logZ = rs->logZ; z.logX = rs->logX;
  z.S_star = rs->S_star; z.remaining = rs->remaining_frac; z.temp_index = rs->index;
  z.done = rs->done;
  *h->h_ctrl = z;
  h->known_done = z.done ? 1 : 0;
  rc = push_ctrl(h);
  if (rc != PHI4_OK) return rc;
  if (h_SE) {
    CU(cudaMemcpyAsync(h->S[c], h_SE, sizeof(float) * N, cudaMemcpyHostToDevice, h->st));
    CU(cudaMemcpyAsync(h->U0[c], h_U0, sizeof(float) * N, cudaMemcpyHostToDevice, h->st));
  } else {
    launch_action(h->phi[c], N, h->ld, h->md, h->S[c], h->U0[c], h->ctrl, h->st);
  }
  if (h->kind == KIND_SMC) {
    h->step_counter = h->step_base = rs->step_counter;
  } else {
    h->iters_enqueued = (uint32_t)(rs->step_counter / (uint64_t)h->n_walk);
    h->iter_base = (int64_t)h->iters_enqueued - (int64_t)rs->index;
  }
  CU(cudaStreamSynchronize(h->st));
  CU(cudaGetLastError());
  return PHI4_OK;
}

PHI4_API int smc_get_chol(phi4smc* h, float* h_Lc) {
  if (!h || !h_Lc) return PHI4_EINVAL;
  CU(cudaStreamSynchronize(h->st));
  CU(cudaMemcpy(h_Lc, h->Lc, sizeof(float) * h->md.V * h->md.V, cudaMemcpyDeviceToHost));
  return PHI4_OK;
}

PHI4_API int smc_set_chol(phi4smc* h, const float* h_Lc) {
  if (!h || !h_Lc) return PHI4_EINVAL;
  CU(cudaMemcpyAsync(h->Lc, h_Lc, sizeof(float) * h->md.V * h->md.V, cudaMemcpyHostToDevice, h->st));
  launch_zero_upper(h->Lc, h->md.V, h->st);
  CU(cudaStreamSynchronize(h->st));
  return PHI4_OK;
}

PHI4_API int smc_get_cov(phi4smc* h, float* h_Sigma) {
  if (!h || !h_Sigma) return PHI4_EINVAL;
  CU(cudaStreamSynchronize(h->st));
  CU(cudaMemcpy(h_Sigma, h->Sigma, sizeof(float) * h->md.V * h->md.V, cudaMemcpyDeviceToHost));
  return PHI4_OK;
}

PHI4_API int smc_get_mean(phi4smc* h, float* h_mu) {
  if (!h || !h_mu) return PHI4_EINVAL;
  CU(cudaStreamSynchronize(h->st));
  CU(cudaMemcpy(h_mu, h->mu, sizeof(float) * h->md.V, cudaMemcpyDeviceToHost));
  return PHI4_OK;
}

PHI4_API int smc_mutate(phi4smc* h, int k, uint8_t* h_accept, float* h_margin) {
  if (!h || h->kind != KIND_SMC || k < 1) return PHI4_EINVAL;
  const bool want = h_accept || h_margin;
  if (want && k > PHI4_MAX_HOOK_STEPS) return PHI4_EINVAL;
  launch_reset_counters(h->ctrl, h->st);
  enqueue_mutation(h, smc_mutate_args(h, k, want ? h->acc_flags : nullptr,
                                      want ? h->margins : nullptr, 0));
  h->step_counter += (uint64_t)k;
  h->step_base += (uint64_t)k;
  const size_t n = (size_t)k * h->N;
  if (h_accept) CU(cudaMemcpyAsync(h_accept, h->acc_flags, n, cudaMemcpyDeviceToHost, h->st));
  if (h_margin) CU(cudaMemcpyAsync(h_margin, h->margins, n * sizeof(float), cudaMemcpyDeviceToHost, h->st));
  launch_reset_counters(h->ctrl, h->st);
  CU(cudaStreamSynchronize(h->st));
  CU(cudaGetLastError());
  return PHI4_OK;
}

PHI4_API int smc_time_mutation(phi4smc* h, int k, int reps, float* h_ms_per_call) {
  if (!h || h->kind != KIND_SMC || k < 1 || reps < 1 || !h_ms_per_call) return PHI4_EINVAL;
  cudaEvent_t e0, e1;
  CU(cudaEventCreate(&e0));
  CU(cudaEventCreate(&e1));
  launch_reset_counters(h->ctrl, h->st);
  CU(cudaEventRecord(e0, h->st));
  for (int r = 0; r < reps; ++r) {
    enqueue_mutation(h, smc_mutate_args(h, k, nullptr, nullptr, 0));
    h->step_counter += (uint64_t)k;
    h->step_base += (uint64_t)k;
  }
  CU(cudaEventRecord(e1, h->st));
  launch_reset_counters(h->ctrl, h->st);
  CU(cudaStreamSynchronize(h->st));
  float ms = 0.f;
  CU(cudaEventElapsedTime(&ms, e0, e1));
  cudaEventDestroy(e0);
  cudaEventDestroy(e1);
  CU(cudaGetLastError());
  *h_ms_per_call = ms / (float)reps;
  return PHI4_OK;
}

// Measurement hook: one phase of the step, `reps` times back to back between two CUDA events on
// the handle's stream.  The state it leaves behind is valid but not meaningful (a proposal that
// was never accepted, a resampling without its reweighting): reset or restore afterwards.
PHI4_API int smc_time_phase(phi4smc* h, int phase, int reps, float* h_ms_per_call) {
  if (!h || h->kind != KIND_SMC || reps < 1 || !h_ms_per_call) return PHI4_EINVAL;
  const int V = h->md.V;
  const bool large = use_tc_propose(h) && !use_tc_path(h);
  if ((phase == PHI4_PHASE_PROPOSAL || phase == PHI4_PHASE_NORMALS || phase == PHI4_PHASE_ACCEPT) && !large)
    return PHI4_EINVAL;
  if (phase < 0 || phase > PHI4_PHASE_REWEIGHT) return PHI4_EINVAL;
  cudaEvent_t e0, e1;
  CU(cudaEventCreate(&e0));
  CU(cudaEventCreate(&e1));
  launch_reset_counters(h->ctrl, h->st);
  MutateArgs a = smc_mutate_args(h, h->prm.k_steps, nullptr, nullptr, 0);
  if (phase == PHI4_PHASE_PROPOSAL || phase == PHI4_PHASE_ACCEPT) {
    // operands of a real step: the factor split and one set of normals, one proposal
    launch_propose_lsplit(a.Lc, V, a.ld, a.s, h->Lsplit, a.ctrl, 0, h->st, a.tc_f16);
    launch_normals_split(a.Z, a.N, a.ld, V, a.seed, a.tag_prop, a.t0, a.ctrl, 0, h->st, a.tc_f16);
    launch_propose_tc(a.phi, a.phip, a.Z, h->Lsplit, a.ld, V, a.ctrl, 0, h->st, a.tc_f16);
  }
  CU(cudaEventRecord(e0, h->st));
  for (int r = 0; r < reps; ++r) {
    switch (phase) {
      case PHI4_PHASE_MUTATION:
        enqueue_mutation(h, smc_mutate_args(h, h->prm.k_steps, nullptr, nullptr, 0));
        h->step_counter += (uint64_t)h->prm.k_steps;
        h->step_base += (uint64_t)h->prm.k_steps;
        break;
      case PHI4_PHASE_PROPOSAL:
        launch_propose_tc(a.phi, a.phip, a.Z, h->Lsplit, a.ld, V, a.ctrl, 0, h->st, a.tc_f16);
        break;
      case PHI4_PHASE_NORMALS:
        launch_normals_split(a.Z, a.N, a.ld, V, a.seed, a.tag_prop, a.t0 + (uint32_t)r, a.ctrl, 0, h->st, a.tc_f16);
        break;
      case PHI4_PHASE_ACCEPT:
        launch_accept_step(a, 0, h->st);
        break;
      case PHI4_PHASE_RESAMPLE:
        enqueue_resample(h);
        break;
      case PHI4_PHASE_GATHER: {
        const int o = h->cur ^ 1;
        launch_gather(h->phi[h->cur], h->phi[o], h->S[h->cur], h->S[o], h->U0[h->cur], h->U0[o], h->anc,
                      nullptr, h->N, h->ld, V, h->ctrl, h->st);
        break;
      }
      case PHI4_PHASE_COVCHOL:
        launch_cov_chol(cov_args(h, 0), h->st);
        break;
      default:   // PHI4_PHASE_REWEIGHT: P1 + P2 at the current beta (beta is put back below)
        launch_next_delta_reweight(h->S[h->cur], h->N, h->prm.ess_target, -1.0, h->w, nullptr, h->ctrl, h->st);
        break;
    }
  }
  CU(cudaEventRecord(e1, h->st));
  launch_reset_counters(h->ctrl, h->st);
  CU(cudaStreamSynchronize(h->st));
  float ms = 0.f;
  CU(cudaEventElapsedTime(&ms, e0, e1));
  cudaEventDestroy(e0);
  cudaEventDestroy(e1);
  CU(cudaGetLastError());
  *h_ms_per_call = ms / (float)reps;
  return PHI4_OK;
}

PHI4_API int smc_reweight(phi4smc* h, double delta, float* h_w, smc_step_info* info) {
  if (!h || h->kind != KIND_SMC) return PHI4_EINVAL;
  launch_next_delta_reweight(h->S[h->cur], h->N, h->prm.ess_target, delta < 0.0 ? -1.0 : delta,
                             h->w, nullptr, h->ctrl, h->st);
  if (h_w) CU(cudaMemcpyAsync(h_w, h->w, sizeof(float) * h->N, cudaMemcpyDeviceToHost, h->st));
  int rc = sync_ctrl(h);
  if (rc == PHI4_ECUDA) return rc;
  if (info) {
    memset(info, 0, sizeof(*info));
    info->beta = h->h_ctrl->beta; info->delta = h->h_ctrl->delta;
    info->ess_frac = h->h_ctrl->ess_frac; info->dlogZ = h->h_ctrl->dlogZ;
    info->logZ = h->h_ctrl->logZ; info->temp_index = h->h_ctrl->temp_index;
    info->done = h->h_ctrl->beta >= 1.0;
  }
  return rc;
}

PHI4_API int smc_resample(phi4smc* h, const float* h_w, int32_t* h_ancestors) {
  if (!h || h->kind != KIND_SMC) return PHI4_EINVAL;
  if (h_w) CU(cudaMemcpyAsync(h->w, h_w, sizeof(float) * h->N, cudaMemcpyHostToDevice, h->st));
  launch_reset_counters(h->ctrl, h->st);
  enqueue_resample(h);
  if (h_ancestors)
    CU(cudaMemcpyAsync(h_ancestors, h->anc, sizeof(int32_t) * h->N, cudaMemcpyDeviceToHost, h->st));
  return sync_ctrl(h);
}
