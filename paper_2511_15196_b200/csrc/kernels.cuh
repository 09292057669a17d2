// kernels.cuh -- host-side launchers of the kernels (one .cu per group), used by api.cu.
// Particles are site-major with a padded stride: phi[x*ld + i], ld = round_up(N,128); the pad
// particles i in [N, ld) hold zeros and never enter a reduction.
#pragma once
#include "common.cuh"

namespace phi4 {

// field.cu -- M1 (INIT stream) and the full action (Eq. 1; U0)
void launch_init_particles(float* phi, int N, int ld, int V, uint64_t seed, cudaStream_t st);
void launch_action(const float* phi, int N, int ld, Model md, float* S, float* U0,
                   Ctrl* ctrl, cudaStream_t st);

void launch_set_identity(float* A, int V, cudaStream_t st);
void launch_zero_upper(float* A, int V, cudaStream_t st);
void launch_reset_counters(Ctrl* ctrl, cudaStream_t st);

// mutate_generic.cu -- M1-M4 for any V, one step = normals -> proposal GEMM -> accept/commit
struct MutateArgs {
  float* phi;        // [V][ld] current particles (updated in place)
  float* phip;       // [V][ld] scratch: proposals
  float* Z;          // [V][ld] scratch: normals
  float* S;          // [ld] cached S_E
  float* U0;         // [ld] cached U0
  const float* Lc;   // [V][V] row-major lower Cholesky factor, strict upper = 0
  Ctrl* ctrl;        // beta / S_star / done are read from here
  uint8_t* acc_out;  // optional [k][N] accept flags
  float* margin_out; // optional [k][N] margins g (R4)
  int N, ld;
  Model md;
  float s;           // step scale
  int mode;          // MODE_SMC / MODE_NS
  uint64_t seed;
  uint32_t tag_prop, tag_acc;
  uint32_t t0;       // step counter of the first step
  int k;             // number of steps
  int respect_done;  // 1: every kernel is a no-op once ctrl->done is set
  // Large-V tcgen05 path only (nullptr otherwise): a second buffer for the split normals, so that the
  // normals of step t+1 are drawn inside the proposal GEMM of step t (they depend on nothing but
  // the counters).
  float* Z2;
  // Fused tcgen05 path only: if set, the last CTA to finish closes the temperature itself
  // (finish_step_device) and the caller launches no finish_step_kernel.
  StepRecord* finish_rec = nullptr;
  int finish_max_rec = 0;
  HostPoll* finish_poll = nullptr;
  // Large-V tcgen05 path: operand format of the split-precision proposal GEMM (propose_tc.cu)
  bool tc_f16 = true;
};
void launch_mutate_generic(const MutateArgs& a, float* Lsplit, cudaStream_t st);
void launch_accept_step(const MutateArgs& a, int j, cudaStream_t st);
// NEXT f3: k constrained slice-sampling steps of the NS walkers (reading A16); a.phip = direction
void launch_ns_slice(const MutateArgs& a, float width, int m_expand, int max_shrink, cudaStream_t st);
// NEXT f2: k independent-MH steps from N(mu, Lc Lc^T) (reading A15); W2 [ld] scratch
bool irmh_supported(int V);
// Lsplit != nullptr: the k steps run in the fused tcgen05 kernel (V <= 112)
void launch_mutate_irmh(const MutateArgs& a, const float* mu, float* W2, float* Lsplit, cudaStream_t st);

// mutate_tc.cu -- M1-M4 fused over k steps on tcgen05 (3xTF32), phi tile resident on-chip
bool mutate_tc_supported(int V, bool irmh = false);
size_t mutate_tc_lsplit_floats(int V);
// mu != nullptr: SMC-IRMH (independent proposal mu + Lc z, W2 = |Lc^-1 (phi - mu)|^2 per particle)
void launch_mutate_tc(const MutateArgs& a, float* Lsplit, cudaStream_t st, const float* mu = nullptr,
                      float* W2 = nullptr);
void launch_lsplit(const float* Lc, int V, int Vn, int Kp, float s, float* Lsplit, const Ctrl* ctrl,
                   int respect_done, cudaStream_t st);

// propose_tc.cu -- M1 + M2 for large V: persistent split-precision tcgen05 GEMM, normals in UMMA
// layout.  f16 = true: 3xFP16 with power-of-two scales (default); false: 3xTF32.
bool propose_tc_supported(int V);
size_t propose_tc_zsplit_floats(int V, int ld);
size_t propose_tc_lsplit_floats(int V);
void propose_tc_dims(int V, int* Vn, int* Kp, bool f16);
// nsteps > 1: steps t .. t + nsteps - 1, one after the other in Zs (propose_tc_zstep_floats apart)
void launch_normals_split(float* Zs, int N, int ld, int V, uint64_t seed, uint32_t tag, uint32_t t,
                          const Ctrl* ctrl, int respect_done, cudaStream_t st, bool f16, int nsteps = 1);
size_t propose_tc_zstep_floats(int V, int ld, bool f16);
int propose_tc_zbatch(int V, int ld, bool f16);
void launch_propose_lsplit(const float* Lc, int V, int ld, float s, float* Lsplit, const Ctrl* ctrl,
                           int respect_done, cudaStream_t st, bool f16);
// next != nullptr: two spare warps of every GEMM CTA also draw the normals of step next->t into
// next->Zs (same layout and numbers as launch_normals_split) while the tensor core works
struct NextNormals { float* Zs; int N; uint64_t seed; uint32_t tag, t; };
void launch_propose_tc(const float* phi, float* phip, const float* Zs, const float* Lsplit, int ld,
                       int V, const Ctrl* ctrl, int respect_done, cudaStream_t st, bool f16,
                       const NextNormals* next = nullptr);

// population.cu -- P1-P4
bool launch_next_delta_reweight(const float* S, int N, float ess_target, double delta_fixed,
                                float* w, unsigned long long* C, Ctrl* ctrl, cudaStream_t st);
void launch_quantise_scan(const float* w, int N, unsigned long long* C, Ctrl* ctrl,
                          cudaStream_t st);
void launch_ancestors(const unsigned long long* C, int N, uint64_t seed, int32_t* anc, uint8_t* flip,
                      int z2, Ctrl* ctrl, cudaStream_t st);
void launch_gather(const float* phi_in, float* phi_out, const float* S_in, float* S_out,
                   const float* U_in, float* U_out, const int32_t* anc, const uint8_t* flip, int N,
                   int ld, int V, Ctrl* ctrl, cudaStream_t st);
void launch_finish_step(Ctrl* ctrl, StepRecord* rec, int max_rec, int k, int N, HostPoll* hp, cudaStream_t st);

// covchol.cu -- C1, C2
struct CovCholArgs {
  const float* phi;  // [V][ld]
  int N, ld, V;
  float* mu;         // [V]
  float* Sigma;      // [V][V]
  float* Lc;         // [V][V]
  float* partial;    // split-K scratch, >= cov_partial_floats(V, N) floats
  float* tc_scratch; // >= syrk_tc_scratch_floats(V, ld) floats, or nullptr: FP32 SIMT syrk
  int tc_small;      // V <= 128: 1 = tcgen05 syrk (syrk_tc_small.cu), 0 = FP32 SIMT reference
  Ctrl* ctrl;
  int respect_done;
  bool tc_f16 = true; // large-V tcgen05 syrk: scaled 3xFP16 operands (false: 3xTF32)
};
size_t cov_partial_floats(int V, int N);
void launch_cov_chol(const CovCholArgs& a, cudaStream_t st);
void launch_cholesky(const float* Sigma, float* Lc, int V, Ctrl* ctrl, int respect_done,
                     cudaStream_t st);

// syrk_tc.cu -- C1 for large V: centred 3xTF32 tcgen05 syrk with K split
bool syrk_tc_supported(int V, int ld);
// syrk_tc_small.cu -- C1 for V <= 128 on tcgen05 (3xTF32), one CTA per 128 particles
bool syrk_tc_small_supported(int V, int ld);
int syrk_tc_small_nsplit(int ld);
void launch_syrk_tc_small(const float* phi, int N, int ld, int V, const float* mu, float* partial,
                          const Ctrl* ctrl, int respect_done, cudaStream_t st);
int syrk_tc_nsplit(int V, int ld, bool f16);
size_t syrk_tc_scratch_floats(int V, int ld);
float* syrk_tc_amax(float* Ps, int V, int ld);     // per-site bounds behind the operand (FP16 scale)
void launch_syrk_tc(const float* phi, int N, int ld, int V, const float* mu, float* Ps,
                    float* partial, const Ctrl* ctrl, int respect_done, cudaStream_t st, bool f16);

// observables.cu -- O
void launch_magnetisation(const float* phi, int N, int ld, int V, float* M, cudaStream_t st);
// out: 5 + 80 doubles (absM, M2, chi, mean_SE, mode_balance, hist); logw may be NULL
void launch_observables_reduce(const float* M, const float* S, const double* logw, int n, int V,
                               double* out, cudaStream_t st);

// ns.cu -- N1-N4
struct NsArgs {
  float* phi; float* S; float* U0;       // live set [V][ld], [ld], [ld]
  float* wphi; float* wS; float* wU;     // walkers [V][ldw], [ldw], [ldw]
  int n, ld, k_del, ldw, V;
  uint64_t seed;
  int32_t* dead;                         // [k_del] by decreasing S_E
  int32_t* surv;                         // [n] survivors in index order
  int32_t* start;                        // [k_del] chosen start points
  float* dead_S; float* dead_M; double* dead_logw;   // dead-point log [max_iters*k_del]
  const double* hsum;                    // [k_del+1] partial sums of 1/(n-m+1) (reading A6), then [k_del] log(1 - e^{-1/(n-j)})
  unsigned long long* gkeys;             // n > 16384: sort keys in global memory (ns_sort_scratch_keys)
  int32_t* gflag;                        // n > 16384: [n] survivor flags
  int max_iters;
  double stop_frac;
  Ctrl* ctrl;
};
size_t ns_sort_scratch_keys(int n);
void launch_ns_hsum(double* hsum, int n, int k_del, cudaStream_t st);
void launch_ns_select_evidence(const NsArgs& a, cudaStream_t st);   // N1 + N2 + start choice
void launch_ns_load_walkers(const NsArgs& a, cudaStream_t st);      // N3 gather
void launch_ns_store_walkers(const NsArgs& a, cudaStream_t st);     // N3 scatter
void launch_ns_finish(const NsArgs& a, StepRecord* rec, int n_walk, HostPoll* hp, cudaStream_t st);  // N4

}  // namespace phi4

namespace phi4 {
// hmc.cu -- NEXT f1: k HMC transitions with mass matrix diag(1/Sigma_xx) (reading A14)
bool hmc_supported(int V);   // the on-chip kernel (L <= 22); larger lattices take launch_hmc_generic
void launch_hmc_generic(float* phi, float* S, float* U0, const float* Sigma, float* q, float* q2,
                        float* p, float* K0, int N, int ld, Model md, float eps, int nfrog, uint64_t seed,
                        uint32_t t0, int k, Ctrl* ctrl, uint8_t* acc_out, float* margin_out,
                        int respect_done, cudaStream_t st);
void launch_hmc(float* phi, float* S, float* U0, const float* Sigma, int N, int ld, Model md,
                float eps, int nfrog, uint64_t seed, uint32_t t0, int k, Ctrl* ctrl,
                uint8_t* acc_out, float* margin_out, int respect_done, cudaStream_t st);
void launch_ns_obs_inputs(const NsArgs& a, int n_dead, float* M_all, float* S_all,
                          double* logw_all, cudaStream_t st);
}
