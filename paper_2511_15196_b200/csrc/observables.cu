// observables.cu -- O: magnetisation observables (reading A13).
#include "kernels.cuh"

namespace phi4 {

// M_i = (1/V) sum_x phi[x][i]; thread per particle, coalesced along i.
__global__ void magnetisation_kernel(const float* __restrict__ phi, int N, int ld, int V,
                                     float* __restrict__ M) {
  int i = blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= N) return;
  float a = 0.f;
  for (int x = 0; x < V; ++x) a += phi[(size_t)x * ld + i];
  M[i] = a / (float)V;
}

void launch_magnetisation(const float* phi, int N, int ld, int V, float* M, cudaStream_t st) {
  ++g_launches; magnetisation_kernel<<<(N + 127) / 128, 128, 0, st>>>(phi, N, ld, V, M);
}

// out[0..4] = <|M|>, <M^2>, chi, <S_E>, mode balance; out[5..84] = normalised weighted histogram
// on [-1.6, 1.6] (80 bins, out-of-range clamped).  Weights exp(logw - max logw), or 1.
__global__ void __launch_bounds__(1024)
observables_reduce_kernel(const float* __restrict__ M, const float* __restrict__ S,
                          const double* __restrict__ logw, int n, int V,
                          double* __restrict__ out) {
  __shared__ double scratch[33];
  __shared__ double hist[80];
  __shared__ double mx_s;
  if (threadIdx.x < 80) hist[threadIdx.x] = 0.0;
  double mx = -INFINITY;
  if (logw) {
    for (int i = threadIdx.x; i < n; i += blockDim.x) mx = fmax(mx, logw[i]);
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) mx = fmax(mx, __shfl_xor_sync(0xffffffffu, mx, o));
    if ((threadIdx.x & 31) == 0) scratch[threadIdx.x >> 5] = mx;
    __syncthreads();
    if (threadIdx.x == 0) {
      double m = -INFINITY;
      for (int k = 0; k < (int)(blockDim.x >> 5); ++k) m = fmax(m, scratch[k]);
      mx_s = m;
    }
    __syncthreads();
    mx = mx_s;
  }
  __syncthreads();
  double W = 0.0, a = 0.0, m2 = 0.0, se = 0.0, npos = 0.0, nneg = 0.0;
  for (int i = threadIdx.x; i < n; i += blockDim.x) {
    double wi = logw ? exp(logw[i] - mx) : 1.0;
    double m = (double)M[i];
    W += wi;
    a += wi * fabs(m);
    m2 += wi * m * m;
    if (S) se += wi * (double)S[i];
    if (m > 0.0) npos += wi; else if (m < 0.0) nneg += wi;   // weight mass per side (reading A19)
    int b = (int)floor((m + 1.6) / (3.2 / 80.0));
    b = b < 0 ? 0 : (b > 79 ? 79 : b);
    atomicAdd(&hist[b], wi);
  }
  W = block_sum(W, scratch);
  a = block_sum(a, scratch);
  m2 = block_sum(m2, scratch);
  se = block_sum(se, scratch);
  npos = block_sum(npos, scratch);
  nneg = block_sum(nneg, scratch);
  __syncthreads();
  if (threadIdx.x == 0) {
    out[0] = a / W;
    out[1] = m2 / W;
    out[2] = (double)V * (out[1] - out[0] * out[0]);
    out[3] = se / W;
    out[4] = nneg > 0.0 ? npos / nneg : INFINITY;
  }
  if (threadIdx.x < 80) out[5 + threadIdx.x] = hist[threadIdx.x] / W;
}

void launch_observables_reduce(const float* M, const float* S, const double* logw, int n, int V,
                               double* out, cudaStream_t st) {
  ++g_launches; observables_reduce_kernel<<<1, 1024, 0, st>>>(M, S, logw, n, V, out);
}

}  // namespace phi4
