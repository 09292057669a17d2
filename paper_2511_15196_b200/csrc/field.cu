// field.cu -- particle initialisation (Philox stream INIT) and the full lattice action.
#include <cstdlib>
#include "kernels.cuh"
#include "philox.cuh"

namespace phi4 {

// phi_i ~ N(0, I): thread (q, i) writes the four sites of quad q of particle i.
__global__ void init_particles_kernel(float* __restrict__ phi, int N, int ld, int V,
                                      uint64_t seed) {
  int i = blockIdx.x * blockDim.x + threadIdx.x;
  int q = blockIdx.y;
  if (i >= ld) return;
  float z[4] = {0.f, 0.f, 0.f, 0.f};
  if (i < N) normals4(seed, TAG_INIT, 0u, (uint32_t)i, (uint32_t)q, z);
#pragma unroll
  for (int j = 0; j < 4; ++j) {
    int x = 4 * q + j;
    if (x < V) phi[(size_t)x * ld + i] = z[j];
  }
}

void launch_init_particles(float* phi, int N, int ld, int V, uint64_t seed, cudaStream_t st) {
  dim3 grid((ld + 127) / 128, (V + 3) / 4);
  ++g_launches; init_particles_kernel<<<grid, 128, 0, st>>>(phi, N, ld, V, seed);
}

// Eq. 1 and U0 for every particle.  A block is 32 particles x 8 row
// groups: warp g sums lattice rows g, g+8, ... of 32 consecutive particles (coalesced 128-byte
// loads in the site-major layout); the 8 partial sums are combined in double.
__global__ void __launch_bounds__(256)
action_kernel(const float* __restrict__ phi, int N, int ld, Model md, float* __restrict__ S,
              float* __restrict__ U0, Ctrl* ctrl) {
  __shared__ float ps[8][32], pu[8][32];
  int lane = threadIdx.x & 31, g = threadIdx.x >> 5;
  int i = blockIdx.x * 32 + lane;
  const int L = md.L;
  float s = 0.f, u = 0.f;
  if (i < N) {
    for (int r = g; r < L; r += 8) {
      int rn = (r + 1 == L) ? 0 : r + 1;
      const float* row = phi + (size_t)r * L * ld + i;
      const float* rown = phi + (size_t)rn * L * ld + i;
      float a = row[0];
      for (int c = 0; c < L; ++c) {
        int cn = (c + 1 == L) ? 0 : c + 1;
        float b = row[(size_t)cn * ld];
        float d = rown[(size_t)c * ld];
        float e = b - a, f = d - a, a2 = a * a;
        s += 0.5f * md.kappa * (e * e + f * f) + a2 * (0.5f * md.m0sq + md.lam * a2);
        u += 0.5f * a2;
        a = b;
      }
    }
  }
  ps[g][lane] = s;
  pu[g][lane] = u;
  __syncthreads();
  if (g == 0 && i < ld) {
    double ts = 0.0, tu = 0.0;
#pragma unroll
    for (int m = 0; m < 8; ++m) { ts += (double)ps[m][lane]; tu += (double)pu[m][lane]; }
    float fs = i < N ? (float)ts : 0.f;
    S[i] = fs;
    U0[i] = i < N ? (float)tu : 0.f;
    if (!isfinite(fs)) ctrl->nan_flag = 1;
  }
}

void launch_action(const float* phi, int N, int ld, Model md, float* S, float* U0, Ctrl* ctrl,
                   cudaStream_t st) {
  ++g_launches; action_kernel<<<ld / 32, 256, 0, st>>>(phi, N, ld, md, S, U0, ctrl);
}

__global__ void set_identity_kernel(float* __restrict__ A, int V) {
  int idx = blockIdx.x * blockDim.x + threadIdx.x;
  if (idx < V * V) A[idx] = (idx / V == idx % V) ? 1.f : 0.f;
}

void launch_set_identity(float* A, int V, cudaStream_t st) {
  ++g_launches; set_identity_kernel<<<(V * V + 255) / 256, 256, 0, st>>>(A, V);
}

// Strict upper triangle := 0 (the proposal GEMM relies on it to stop each tile at its last row).
__global__ void zero_upper_kernel(float* __restrict__ A, int V) {
  int idx = blockIdx.x * blockDim.x + threadIdx.x;
  if (idx < V * V && (idx % V) > (idx / V)) A[idx] = 0.f;
}

void launch_zero_upper(float* A, int V, cudaStream_t st) {
  ++g_launches; zero_upper_kernel<<<(V * V + 255) / 256, 256, 0, st>>>(A, V);
}

__global__ void reset_counters_kernel(Ctrl* ctrl) { ctrl->n_accept = 0u; ctrl->n_unique = 0u; }
bool pdl_enabled() {
  static const bool on = [] { const char* e = getenv("PHI4_NO_PDL"); return !(e && e[0] == '1'); }();
  return on;
}

void launch_reset_counters(Ctrl* ctrl, cudaStream_t st) {
  ++g_launches; reset_counters_kernel<<<1, 1, 0, st>>>(ctrl);
}

}  // namespace phi4
