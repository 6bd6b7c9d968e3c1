// static_scratch.cu -- gwmf_power_table_static: the Eq. 4 power table C[k] computed with NO device allocation at all.
//
// Who this is for.  Everything else in the library works out of a workspace the caller allocates (gwmf_create).  Some
// callers cannot get one at the moment they need the table:
//   * a low-latency online search refreshes its PSD estimate every few seconds while filters run; cudaMalloc / cudaFree
//     take a device-wide lock and may wait for all running work, which stalls those filters for an unbounded time;
//   * a host process in which another component (a framework's caching allocator, a second pipeline) has already
//     reserved the card's memory: a fresh cudaMalloc fails or fragments the pool;
//   * plug-in code that is handed input and output buffers by its host and is not allowed to own device memory.
// For them the scratch of this one operation lives INSIDE the library image: a file-scope __device__ array of
// GWMF_STATIC_SCRATCH_BYTES (8448) bytes.  Every GPU on which the library's device code gets loaded holds that array
// until the process exits; that is the price, and the reason the maximum is small and fixed.
//
// What it computes: the same table gwmf_load_segment builds in its workspace (segment.cu: k_power_terms, k_prefix_*):
//   g[k] = f_k^(-7/3) / S_n[k] for k_low <= k < n/2 (0 below),   C[k] = sum_{k' <= k} g[k']        (Eq. 4)
// in the same fixed summation order (1024 contiguous chunks, each summed front to back, chunk totals scanned front to
// back), so the result is bit-identical to the workspace path's; sigma^2 = 4 df C[k_high - 1] and the equal-power band
// edges follow from it.  The variant differs from the workspace kernels in two ways: g[k] is evaluated
// inside the two prefix kernels instead of being staged in an n/2-entry table (so the scratch is the 1024 chunk totals
// and one status word, whatever n), and those live in the static array.
//
// About the array's name.  In HOST code `g_static_scratch` is only a handle the runtime uses to look the symbol up; it
// is not a device address and must never be handed to a kernel or to cudaMemset as if it were.  The device address is
// obtained once per device, with that device current, from cudaGetSymbolAddress (resolve_scratch below) and it is that
// pointer the kernels receive.
#include <mutex>
#include <stdio.h>

#include "gwmf_internal.cuh"

namespace {

constexpr int kChunks = 1024;                          // same cut as segment.cu: kPrefixChunks
constexpr size_t kTotalsBytes = kChunks * sizeof(double);
constexpr size_t kStatusOff = kTotalsBytes;            // one int32: 1 if S_n was not finite and > 0 inside the band
constexpr size_t kScratchBytes = kTotalsBytes + 256;
static_assert(kScratchBytes == GWMF_STATIC_SCRATCH_BYTES, "include/gwmf.h states the size of the built-in scratch");

// The scratch itself.  One per device that loads this library, shared by every call on that device.
static __device__ __align__(256) unsigned char g_static_scratch[kScratchBytes];

// Integrand of Eq. 4 at bin k, the arithmetic of k_tables (u = f^(-1/3)) and k_power_terms (u^7 / S_n) verbatim.
__device__ __forceinline__ double power_term(const double* __restrict__ sn, int k, int k_low, double df, int* bad) {
  if (k < k_low) return 0.0;
  const double S = sn[k];
  if (!(S > 0.0) || isinf(S)) {
    atomicOr(bad, 1);
    return 0.0;
  }
  const double u = rcbrt((double)k * df), u2 = u * u, u4 = u2 * u2;
  return u4 * u2 * u / S;
}

// One warp per chunk of L bins: the terms go to shared memory with coalesced loads of S_n, lane 0 adds them front to back.
__global__ void __launch_bounds__(32) k_st_totals(const double* __restrict__ sn, double* __restrict__ totals, int* bad,
                                                  int half_n, int L, int k_low, double df) {
  extern __shared__ double sh[];
  const int lo = blockIdx.x * L, hi = min(lo + L, half_n);
  for (int k = lo + threadIdx.x; k < hi; k += 32) sh[k - lo] = power_term(sn, k, k_low, df, bad);
  __syncwarp();
  if (threadIdx.x == 0) {
    double acc = 0.0;
    for (int k = 0; k < hi - lo; ++k) acc += sh[k];
    totals[blockIdx.x] = acc;                          // every one of the 1024 entries is written by every call
  }
}

__global__ void k_st_scan(double* __restrict__ totals) {                 // exclusive, front to back
  double run = 0.0;
  for (int i = 0; i < kChunks; ++i) { const double v = totals[i]; totals[i] = run; run += v; }
}

__global__ void __launch_bounds__(32) k_st_write(const double* __restrict__ sn, const double* __restrict__ offsets,
                                                 double* __restrict__ c_tab, int* bad, int half_n, int L, int k_low, double df) {
  extern __shared__ double sh[];
  const int lo = blockIdx.x * L, hi = min(lo + L, half_n);
  for (int k = lo + threadIdx.x; k < hi; k += 32) sh[k - lo] = power_term(sn, k, k_low, df, bad);
  __syncwarp();
  if (threadIdx.x == 0) {
    double acc = offsets[blockIdx.x];
    for (int k = 0; k < hi - lo; ++k) { acc += sh[k]; sh[k] = acc; }
  }
  __syncwarp();
  for (int k = lo + threadIdx.x; k < hi; k += 32) c_tab[k] = sh[k - lo];
}

// Device address of g_static_scratch on each device, resolved on the first call made with that device current.
constexpr int kMaxDevices = 64;
std::mutex g_mu;
unsigned char* g_scratch_addr[kMaxDevices];            // nullptr = not resolved yet

cudaError_t resolve_scratch(int dev, unsigned char** out) {
  std::lock_guard<std::mutex> lock(g_mu);
  if (!g_scratch_addr[dev]) {
    int major = 0;
    cudaError_t e = cudaDeviceGetAttribute(&major, cudaDevAttrComputeCapabilityMajor, dev);
    if (e != cudaSuccess) return e;
    if (major < 10) return cudaErrorNoKernelImageForDevice;            // sm_100a code only, as gwmf_create
    void* p = nullptr;
    e = cudaGetSymbolAddress(&p, g_static_scratch);                    // `dev` is the current device here
    if (e != cudaSuccess) return e;
    if (!p) return cudaErrorInvalidSymbol;
    g_scratch_addr[dev] = static_cast<unsigned char*>(p);
  }
  *out = g_scratch_addr[dev];
  return cudaSuccess;
}

int fail(int status, char* err, size_t err_len, const char* fmt, long long a = 0, long long b = 0) {
  if (err && err_len) snprintf(err, err_len, fmt, a, b);
  return status;
}

int fail_cuda(cudaError_t e, char* err, size_t err_len, const char* where) {
  if (err && err_len) snprintf(err, err_len, "%s: %s", where, cudaGetErrorString(e));
  return GWMF_E_CUDA;
}

}  // namespace

extern "C" int gwmf_power_table_static(const double* d_sn, double* d_c, int64_t n, double fs, double f_low,
                                       void* cuda_stream, char* err, size_t err_len) {
  if (err && err_len) err[0] = '\0';
  if (!d_sn || !d_c) return fail(GWMF_E_ARG, err, err_len, "gwmf_power_table_static: null S_n or C pointer");
  if (n > GWMF_STATIC_MAX_N)
    return fail(GWMF_E_CAPACITY, err, err_len,
                "gwmf_power_table_static: n = %lld is beyond the %lld samples the built-in scratch is laid out for; "
                "use gwmf_create / gwmf_load_segment with a workspace of your own", (long long)n, (long long)GWMF_STATIC_MAX_N);
  if (n < (1 << 14) || (n & (n - 1)) != 0)
    return fail(GWMF_E_ARG, err, err_len, "gwmf_power_table_static: n = %lld is not a power of two >= 2^14", (long long)n);
  if (!(fs > 0.0) || !(f_low > 0.0) || !(f_low < 0.5 * fs))
    return fail(GWMF_E_ARG, err, err_len, "gwmf_power_table_static: need 0 < f_low < fs / 2");
  int dev = -1;
  cudaError_t e = cudaGetDevice(&dev);
  if (e != cudaSuccess) return fail_cuda(e, err, err_len, "cudaGetDevice");
  if (dev < 0 || dev >= kMaxDevices)
    return fail(GWMF_E_ARG, err, err_len, "gwmf_power_table_static: device ordinal %lld is outside 0..%lld", dev, kMaxDevices - 1);
  unsigned char* scratch = nullptr;
  if ((e = resolve_scratch(dev, &scratch)) != cudaSuccess) return fail_cuda(e, err, err_len, "cudaGetSymbolAddress(static scratch)");
  double* totals = reinterpret_cast<double*>(scratch);
  int* bad = reinterpret_cast<int*>(scratch + kStatusOff);
  cudaStream_t st = static_cast<cudaStream_t>(cuda_stream);
  const int half = (int)(n / 2);
  const double df = fs / (double)n;
  const int k_low = (int)ceil(f_low / df);
  const int L = (half + kChunks - 1) / kChunks;
  const size_t sm = (size_t)L * sizeof(double);        // 16 KB at n = 2^22: inside the 48 KB every kernel may use
  // The array keeps what the previous call left in it.  The chunk totals are all rewritten before they are read; the
  // status word is OR-ed into, so it is the one thing that has to start at zero.
  if ((e = cudaMemsetAsync(bad, 0, sizeof(int), st)) != cudaSuccess) return fail_cuda(e, err, err_len, "cudaMemsetAsync(status)");
  k_st_totals<<<kChunks, 32, sm, st>>>(d_sn, totals, bad, half, L, k_low, df);
  k_st_scan<<<1, 1, 0, st>>>(totals);
  k_st_write<<<kChunks, 32, sm, st>>>(d_sn, totals, d_c, bad, half, L, k_low, df);
  if ((e = cudaGetLastError()) != cudaSuccess) return fail_cuda(e, err, err_len, "kernel launch");
  int h_bad = 0;
  if ((e = cudaMemcpyAsync(&h_bad, bad, sizeof(int), cudaMemcpyDeviceToHost, st)) != cudaSuccess)
    return fail_cuda(e, err, err_len, "cudaMemcpyAsync(status)");
  if ((e = cudaStreamSynchronize(st)) != cudaSuccess) return fail_cuda(e, err, err_len, "cudaStreamSynchronize");
  if (h_bad)
    return fail(GWMF_E_ARG, err, err_len, "gwmf_power_table_static: S_n has an entry inside [f_low, fs/2) that is not finite and > 0");
  return GWMF_OK;
}
