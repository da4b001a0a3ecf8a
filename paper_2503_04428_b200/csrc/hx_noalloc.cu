// hx_noalloc.cu -- hx_self_gravity_noalloc: the self-gravity refresh (Eq. 4; R28) as an entry
// point that allocates NOTHING, for callers that cannot call cudaMalloc (CUDA graph capture, tight serving loops, harnesses
// that forbid it).  It is a variant of the shell-mass reduction + scan of hx_aux.cu (shell_mass_partial_kernel,
// self_gravity_table_kernel), whose scratch -- the partial shell sums [groups][n0] and the angular weights [n1 + n2] -- lives
// in a handle's cudaMalloc'ed memory there and in a file-scope `static __device__` array here.
//
// The array has a fixed, modest size (2 MiB + 32 KiB); every GPU that loads the library holds it until the process exits.
// In HOST code its name is a host-side stand-in, not a device address: the kernels get the address cudaGetSymbolAddress returns,
// resolved once per device with that device current.  Every call on a GPU shares the array: it keeps the last call's contents
// (each call writes every entry it later reads, so nothing has to start at zero), and calls that overlap on the GPU race.
#include <cstdio>
#include <mutex>

#include "hx_common.cuh"

namespace {

constexpr int NA_GROUPS = 128;                                   // row groups of the shell-mass reduction
constexpr size_t NA_PARTIAL = (size_t)NA_GROUPS * HX_NOALLOC_MAX_N0;   // doubles: partial shell sums [group][n0]
constexpr size_t NA_TOTAL = NA_PARTIAL + HX_NOALLOC_MAX_ANGULAR;       // + theta weights [n1], phi widths [n2]
constexpr int NA_MAX_DEVICES = 64;

static __device__ __align__(256) double g_noalloc_scratch[NA_TOTAL];   // 2 MiB + 32 KiB per GPU

// angular weights: cos(th-) - cos(th+) per theta cell, phi width per phi cell
__global__ void na_weights_kernel(const double* __restrict__ ft, const double* __restrict__ fp, int n1, int n2, double* __restrict__ w) {
  const int t = blockIdx.x * blockDim.x + threadIdx.x;
  if (t < n1) w[t] = cos(ft[t]) - cos(ft[t + 1]);
  else if (t < n1 + n2) w[t] = fp[t - n1 + 1] - fp[t - n1];
}

// stage 1: block (bx, group) sums rho x (theta weight) x (phi weight) over the rows group, group + groups, ... for 256 radial
// cells (coalesced along r) and writes ONE entry per (group, i): every entry stage 2 reads is written here, in this call
__global__ void na_partial_kernel(const double* __restrict__ rho, int n0, int n1, int n2, const double* __restrict__ w, double* __restrict__ partial) {
  const int i = blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= n0) return;
  const int rows = n1 * n2;
  double acc = 0.0;
  for (int r = blockIdx.y; r < rows; r += gridDim.y) {
    const int j = r % n1, k = r / n1;
    acc = fma(rho[(size_t)r * n0 + i], w[j] * w[n1 + k], acc);
  }
  partial[(size_t)blockIdx.y * n0 + i] = acc;
}

// stage 2: one block adds the partial sums in group order (deterministic), scans over r and writes g[0 .. n0-1]
__global__ void na_table_kernel(const double* __restrict__ partial, int groups, const double* __restrict__ fr, const double* __restrict__ ft,
                                const double* __restrict__ fp, int n0, int n1, int n2, double GM, double G, double* __restrict__ g) {
  extern __shared__ double m[];             // shell masses [n0]
  for (int i = threadIdx.x; i < n0; i += blockDim.x) {
    double s = 0.0;
    for (int b = 0; b < groups; ++b) s += partial[(size_t)b * n0 + i];
    const double rm = fr[i], rp = fr[i + 1];
    m[i] = s * ((rp * rp * rp - rm * rm * rm) / 3.0);
  }
  __syncthreads();
  if (threadIdx.x == 0) {
    const double PI = 3.14159265358979323846;
    const double domega = (cos(ft[0]) - cos(ft[n1])) * (fp[n2] - fp[0]);
    const double scale = G * 4.0 * PI / domega;
    double below = 0.0;
    for (int i = 0; i < n0; ++i) {
      const double rm = fr[i], rp = fr[i + 1], rc = 0.5 * (rm + rp);
      const double frac = (rc * rc * rc - rm * rm * rm) / (rp * rp * rp - rm * rm * rm);
      g[i] = -(GM + scale * (below + m[i] * frac)) / (rc * rc);
      below += m[i];
    }
  }
}

thread_local char t_err[256] = {0};

int na_fail(int code, const char* fmt, long long a = 0, long long b = 0) {
  snprintf(t_err, sizeof(t_err), fmt, a, b);
  return code;
}

// Device address of the scratch array on the CURRENT device: cudaGetSymbolAddress once per device, with that device current.
cudaError_t scratch_address(double** out) {
  static std::mutex mu;
  static double* addr[NA_MAX_DEVICES] = {nullptr};
  int dev = 0;
  cudaError_t e = cudaGetDevice(&dev);
  if (e != cudaSuccess) return e;
  if (dev < 0 || dev >= NA_MAX_DEVICES) return cudaErrorInvalidDevice;
  std::lock_guard<std::mutex> lock(mu);
  if (!addr[dev]) {
    double* p = nullptr;
    e = cudaGetSymbolAddress((void**)&p, g_noalloc_scratch);
    if (e != cudaSuccess) return e;
    if (!p) return cudaErrorInvalidSymbol;
    addr[dev] = p;
  }
  *out = addr[dev];
  return cudaSuccess;
}

}  // namespace

extern "C" {

const char* hx_noalloc_error(void) { return t_err; }

int hx_self_gravity_noalloc(const double* rho, const double* faces_r, const double* faces_theta, const double* faces_phi, int n0, int n1,
                            int n2, double GM, double G, double* g, void* cuda_stream) {
  t_err[0] = 0;
  if (!rho || !faces_r || !faces_theta || !faces_phi || !g) return na_fail(HX_ERR_INVALID_ARG, "hx_self_gravity_noalloc: null pointer");
  if (n0 < 1 || n1 < 1 || n2 < 1) return na_fail(HX_ERR_INVALID_ARG, "hx_self_gravity_noalloc: n0, n1, n2 must be >= 1");
  if (n0 > HX_NOALLOC_MAX_N0)
    return na_fail(HX_ERR_UNSUPPORTED, "hx_self_gravity_noalloc: n0 = %lld exceeds HX_NOALLOC_MAX_N0 = %lld (fixed static scratch array)", n0,
                   HX_NOALLOC_MAX_N0);
  if ((long long)n1 + n2 > HX_NOALLOC_MAX_ANGULAR)
    return na_fail(HX_ERR_UNSUPPORTED, "hx_self_gravity_noalloc: n1 + n2 = %lld exceeds HX_NOALLOC_MAX_ANGULAR = %lld (fixed static scratch array)",
                   (long long)n1 + n2, HX_NOALLOC_MAX_ANGULAR);
  double* scratch = nullptr;
  cudaError_t e = scratch_address(&scratch);
  if (e != cudaSuccess) {
    snprintf(t_err, sizeof(t_err), "hx_self_gravity_noalloc: scratch address: %s", cudaGetErrorString(e));
    return HX_ERR_CUDA;
  }
  double* partial = scratch;
  double* weights = scratch + NA_PARTIAL;
  cudaStream_t st = (cudaStream_t)cuda_stream;
  const long long rows = (long long)n1 * n2;
  const int groups = (int)(rows < NA_GROUPS ? rows : NA_GROUPS);
  na_weights_kernel<<<(n1 + n2 + 255) / 256, 256, 0, st>>>(faces_theta, faces_phi, n1, n2, weights);
  na_partial_kernel<<<dim3((unsigned)((n0 + 255) / 256), (unsigned)groups), 256, 0, st>>>(rho, n0, n1, n2, weights, partial);
  na_table_kernel<<<1, 256, (size_t)n0 * sizeof(double), st>>>(partial, groups, faces_r, faces_theta, faces_phi, n0, n1, n2, GM, G, g);   // <= 16 KiB
  e = cudaGetLastError();
  if (e != cudaSuccess) {
    snprintf(t_err, sizeof(t_err), "hx_self_gravity_noalloc: launch: %s", cudaGetErrorString(e));
    return HX_ERR_CUDA;
  }
  return HX_OK;
}

}  // extern "C"
