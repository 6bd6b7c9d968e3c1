// probe.cu -- measurement helper: the FP32 (non-tensor) peak of the device the way the hot kernels use the pipe,
// i.e. chains of packed fma.rn.f32x2 (FFMA2).  bench.py reports it beside the derived figure
// (SMs x 128 lanes x 2 flop x clock) for the "alu" roofline of the spill-free path.
#include "fft_reg.cuh"
#include "gwmf_internal.cuh"

namespace gwmf {

constexpr int kProbeChains = 8;
constexpr int kProbeIters = 4096;

__global__ void __launch_bounds__(256) k_fma_probe(float2* __restrict__ out, float seed) {
  pk2 acc[kProbeChains];
#pragma unroll
  for (int i = 0; i < kProbeChains; ++i) acc[i] = pk(seed + (float)i, seed - (float)(threadIdx.x & 7));
  const pk2 a = pk(0.999f, 1.001f), b = pk(1e-3f, -1e-3f);
#pragma unroll 1
  for (int it = 0; it < kProbeIters; it += 4) {
#pragma unroll
    for (int u = 0; u < 4; ++u)
#pragma unroll
      for (int i = 0; i < kProbeChains; ++i) acc[i] = fma2(acc[i], a, b);       // 8 independent chains per thread
  }
  float2 s = make_float2(0.f, 0.f);
#pragma unroll
  for (int i = 0; i < kProbeChains; ++i) s = cadd(s, unpk(acc[i]));
  if (s.x == 123.456f) out[blockIdx.x * blockDim.x + threadIdx.x] = s;          // never true: keeps the chains alive
}

}  // namespace gwmf

extern "C" int gwmf_fma_peak(void* cuda_stream, int32_t repeats, double* host_tflops) {
  using namespace gwmf;
  if (!host_tflops || repeats < 1) return GWMF_E_ARG;
  cudaStream_t st = (cudaStream_t)cuda_stream;
  int dev = 0, sms = 0;
  if (cudaGetDevice(&dev) != cudaSuccess || cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess)
    return GWMF_E_CUDA;
  float2* d_out = nullptr;
  const int blocks = sms * 8;
  if (cudaMalloc((void**)&d_out, sizeof(float2) * (size_t)blocks * 256) != cudaSuccess) return GWMF_E_CUDA;
  cudaEvent_t e0, e1;
  cudaEventCreate(&e0);
  cudaEventCreate(&e1);
  double best = 0.0;
  for (int r = 0; r < repeats + 1; ++r) {                  // the first launch is the warm-up
    cudaEventRecord(e0, st);
    k_fma_probe<<<blocks, 256, 0, st>>>(d_out, 1.0f + (float)r);
    cudaEventRecord(e1, st);
    if (cudaEventSynchronize(e1) != cudaSuccess) { best = -1.0; break; }
    float ms = 0.f;
    cudaEventElapsedTime(&ms, e0, e1);
    const double flop = (double)blocks * 256.0 * (double)kProbeIters * kProbeChains * 4.0;   // FFMA2 = 2 lanes x 2 flop
    if (r > 0 && ms > 0.f && flop / (ms * 1e-3) / 1e12 > best) best = flop / (ms * 1e-3) / 1e12;
  }
  cudaEventDestroy(e0);
  cudaEventDestroy(e1);
  cudaFree(d_out);
  if (best <= 0.0) return GWMF_E_CUDA;
  *host_tflops = best;
  return GWMF_OK;
}
