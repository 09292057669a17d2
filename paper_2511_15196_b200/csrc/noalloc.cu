// noalloc.cu -- phi4_resample_noalloc: exact systematic resampling (P3; reading R5) for
// callers that cannot allocate device memory (code under CUDA graph capture, tight serving loops,
// harnesses that forbid cudaMalloc).  The caller passes the weights and receives the ancestors;
// the kernels' scratch -- the 64-bit integer CDF, the block sums of the multi-block scan, the flip
// bytes and a control block -- lives in ONE file-scope __device__ array of fixed size, so the call
// allocates nothing: no cudaMalloc / cudaFree, no allocating library routine, no workspace.
//
// Cost: every GPU that loads libphi4smc.so holds PHI4_NOALLOC_SCRATCH_BYTES (about 1.2 MB) until
// the process exits, whether or not this entry point is ever called.
//
// The array is shared by every call and keeps the last call's contents.  The control block is
// re-initialised by a kernel at the start of each call (everything else is fully overwritten for
// the N entries a call uses before it is read), so stale contents never enter a result.  Calls
// that overlap on the GPU (two streams, two host threads) RACE on the array: serialise them.
//
// In host code `g_noalloc_scratch` is a host-side stand-in, not a device address.  The device
// address is taken once per device with cudaGetSymbolAddress (that device current) and only that
// pointer is handed to kernels; device code (noalloc_prepare_kernel) names the array directly.
#include <mutex>

#include "../../include/phi4smc.h"
#include "kernels.cuh"

namespace phi4 {

constexpr int NA_MAX_N = PHI4_NOALLOC_MAX_N;
// layout (bytes): [0, 256) control block | CDF: (NA_MAX_N + 256) x 8 (the + 256: block sums of the
// two-launch scan, as launch_quantise_scan expects behind round_up(N, 128) entries) | flips: NA_MAX_N
constexpr size_t NA_OFF_CTRL = 0;
constexpr size_t NA_OFF_CDF = 256;
constexpr size_t NA_OFF_FLIP = NA_OFF_CDF + (size_t)(NA_MAX_N + 256) * sizeof(unsigned long long);
constexpr size_t NA_BYTES = NA_OFF_FLIP + (size_t)NA_MAX_N;
static_assert(sizeof(Ctrl) <= 256, "control block must fit its slot");
static_assert(NA_BYTES <= PHI4_NOALLOC_SCRATCH_BYTES, "header constant out of date");
static_assert(NA_OFF_FLIP % 256 == 0, "sub-arrays stay 256-byte aligned");

static __device__ __align__(256) unsigned char g_noalloc_scratch[PHI4_NOALLOC_SCRATCH_BYTES];

// Device code may name the array directly.  Fresh control block for one resampling: not done, no
// NaN flag, q_total = 0 until the scan writes it, temp_index = t (keys the RESAMPLE stream, R1).
__global__ void noalloc_prepare_kernel(uint32_t t) {
  if (blockIdx.x != 0 || threadIdx.x != 0) return;
  Ctrl* c = reinterpret_cast<Ctrl*>(g_noalloc_scratch + NA_OFF_CTRL);
  Ctrl z = {};
  z.temp_index = (int)t;
  *c = z;
}

namespace {
constexpr int NA_MAX_DEVICES = 64;
unsigned char* g_dev_ptr[NA_MAX_DEVICES] = {};      // device address of the array, per device
std::mutex g_mu;

// Device address of the scratch array on the CURRENT device (looked up once per device).
int scratch_address(unsigned char** out) {
  int dev = -1;
  if (cudaGetDevice(&dev) != cudaSuccess || dev < 0 || dev >= NA_MAX_DEVICES) return PHI4_ECUDA;
  std::lock_guard<std::mutex> lk(g_mu);
  if (!g_dev_ptr[dev]) {
    void* p = nullptr;
    if (cudaGetSymbolAddress(&p, g_noalloc_scratch) != cudaSuccess || !p) {
      cudaGetLastError();
      return PHI4_ECUDA;
    }
    g_dev_ptr[dev] = static_cast<unsigned char*>(p);
  }
  *out = g_dev_ptr[dev];
  return PHI4_OK;
}
}  // namespace

}  // namespace phi4

using namespace phi4;

#define PHI4_API extern "C" __attribute__((visibility("default")))

PHI4_API int phi4_noalloc_setup(void) {
  unsigned char* p = nullptr;
  return scratch_address(&p);
}

PHI4_API int phi4_resample_noalloc(const float* d_w, int N, uint64_t seed, uint32_t t,
                                   int32_t* d_ancestors, void* cuda_stream) {
  if (!d_w || !d_ancestors || N < 1) return PHI4_EINVAL;
  if (N > NA_MAX_N) return PHI4_ETOOBIG;
  unsigned char* base = nullptr;
  int rc = scratch_address(&base);
  if (rc != PHI4_OK) return rc;
  cudaStream_t st = reinterpret_cast<cudaStream_t>(cuda_stream);
  Ctrl* ctrl = reinterpret_cast<Ctrl*>(base + NA_OFF_CTRL);
  unsigned long long* C = reinterpret_cast<unsigned long long*>(base + NA_OFF_CDF);
  uint8_t* flip = base + NA_OFF_FLIP;
  ++g_launches; noalloc_prepare_kernel<<<1, 32, 0, st>>>(t);
  launch_quantise_scan(d_w, N, C, ctrl, st);                       // q_i = floor(w_i 2^40), integer CDF
  launch_ancestors(C, N, seed, d_ancestors, flip, 0, ctrl, st);    // a_j = #{i : C_i <= t_j}
  return cudaGetLastError() == cudaSuccess ? PHI4_OK : PHI4_ECUDA;
}
