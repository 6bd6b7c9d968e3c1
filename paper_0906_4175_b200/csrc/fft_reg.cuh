// fft_reg.cuh -- in-register complex FFTs of R = 2..32 points (one thread owns all R points).
//
// Inverse sign: X[k] = sum_n x[n] e^{+2 pi i nk/R}, the e^{2 pi i f t} of Eq. 1.
// Decimation in frequency, radix 2, all loops unrolled so that every twiddle is a compile-time
// constant and trivial factors (1, i, (1+-i)/sqrt 2) cost no multiplies.  The result is left in
// bit-reversed order: X[k] is in x[brev<R>(k)].
#pragma once
#include <cuda_runtime.h>

namespace gwmf {

// cos(2 pi q / 32), q = 0..8, correctly rounded from fp64
__host__ __device__ constexpr double cos32_tab(int q) {
  return q == 0 ? 1.0
       : q == 1 ? 0.98078528040323044913
       : q == 2 ? 0.92387953251128675613
       : q == 3 ? 0.83146961230254523708
       : q == 4 ? 0.70710678118654752440
       : q == 5 ? 0.55557023301960222474
       : q == 6 ? 0.38268343236508977173
       : q == 7 ? 0.19509032201612826785
       : 0.0;
}
// cos / sin of 2 pi q / 32 for any q in [0, 32)
__host__ __device__ constexpr double cos32(int q) {
  q &= 31;
  return q <= 8 ? cos32_tab(q) : q <= 16 ? -cos32_tab(16 - q) : q <= 24 ? -cos32_tab(q - 16) : cos32_tab(32 - q);
}
__host__ __device__ constexpr double sin32(int q) { return cos32(q - 8); }

template <int R>
__host__ __device__ constexpr int brev(int k) {
  int r = 0;
  for (int b = 1; b < R; b <<= 1) { r = (r << 1) | (k & 1); k >>= 1; }
  return r;
}

__device__ __forceinline__ float2 cmul(float2 a, float2 b) {
  return make_float2(fmaf(a.x, b.x, -a.y * b.y), fmaf(a.x, b.y, a.y * b.x));
}
__device__ __forceinline__ float2 cadd(float2 a, float2 b) { return make_float2(a.x + b.x, a.y + b.y); }
__device__ __forceinline__ float2 csub(float2 a, float2 b) { return make_float2(a.x - b.x, a.y - b.y); }

// d * e^{+2 pi i Q/32} with Q a compile-time constant
template <int Q>
__device__ __forceinline__ float2 mul_w32(float2 d) {
  constexpr int q = Q & 31;
  if constexpr (q == 0) return d;
  else if constexpr (q == 8) return make_float2(-d.y, d.x);
  else if constexpr (q == 16) return make_float2(-d.x, -d.y);
  else if constexpr (q == 24) return make_float2(d.y, -d.x);
  else if constexpr (q == 4) { constexpr float h = (float)cos32_tab(4); return make_float2(h * (d.x - d.y), h * (d.x + d.y)); }
  else if constexpr (q == 12) { constexpr float h = (float)cos32_tab(4); return make_float2(-h * (d.x + d.y), h * (d.x - d.y)); }
  else if constexpr (q == 20) { constexpr float h = (float)cos32_tab(4); return make_float2(-h * (d.x - d.y), -h * (d.x + d.y)); }
  else if constexpr (q == 28) { constexpr float h = (float)cos32_tab(4); return make_float2(h * (d.x + d.y), -h * (d.x - d.y)); }
  else {
    constexpr float c = (float)cos32(q), s = (float)sin32(q);
    return make_float2(fmaf(d.x, c, -d.y * s), fmaf(d.x, s, d.y * c));
  }
}

template <int R, int H, int BASE, int M>
struct DifInner {
  __device__ __forceinline__ static void run(float2 (&x)[R]) {
    if constexpr (M < H) {
      float2 a = x[BASE + M], b = x[BASE + M + H];
      x[BASE + M] = cadd(a, b);
      x[BASE + M + H] = mul_w32<M * (16 / H)>(csub(a, b));   // W_{2H}^M = W_32^{M*32/(2H)}
      DifInner<R, H, BASE, M + 1>::run(x);
    }
  }
};
template <int R, int H, int BASE>
struct DifBlocks {
  __device__ __forceinline__ static void run(float2 (&x)[R]) {
    if constexpr (BASE < R) {
      DifInner<R, H, BASE, 0>::run(x);
      DifBlocks<R, H, BASE + 2 * H>::run(x);
    }
  }
};
template <int R, int H>
struct DifStages {
  __device__ __forceinline__ static void run(float2 (&x)[R]) {
    if constexpr (H >= 1) {
      DifBlocks<R, H, 0>::run(x);
      DifStages<R, H / 2>::run(x);
    }
  }
};

// In place; afterwards X[k] = x[brev<R>(k)].  R in {1, 2, 4, 8, 16, 32}.
template <int R>
__device__ __forceinline__ void fft_dif(float2 (&x)[R]) {
  static_assert(R >= 1 && R <= 32 && (R & (R - 1)) == 0, "R must be a power of two <= 32");
  DifStages<R, R / 2>::run(x);
}

}  // namespace gwmf
