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

// ---- packed fp32x2 arithmetic (sm_100: FFMA2 / FADD2 / FMUL2 work on an aligned register pair) ------------
// A complex number (re, im) is one packed operand, so a complex add is ONE instruction and a butterfly with
// a general twiddle THREE (see bfly_w32).  ptxas folds the half swap (.LO_HI), the negation of one half
// (.NP) and of both halves into operand modifiers, and takes compile-time constants as immediates.  The
// FMA pipe does the same work per flop as with scalar FFMA; what is halved is the issue-slot count.
typedef unsigned long long pk2;
__device__ __forceinline__ pk2 pk(float lo, float hi) { pk2 r; asm("mov.b64 %0, {%1, %2};" : "=l"(r) : "f"(lo), "f"(hi)); return r; }
__device__ __forceinline__ pk2 pk(float2 v) { return pk(v.x, v.y); }
__device__ __forceinline__ float2 unpk(pk2 v) { float2 r; asm("mov.b64 {%0, %1}, %2;" : "=f"(r.x), "=f"(r.y) : "l"(v)); return r; }
__device__ __forceinline__ pk2 fma2(pk2 a, pk2 b, pk2 c) { pk2 r; asm("fma.rn.f32x2 %0, %1, %2, %3;" : "=l"(r) : "l"(a), "l"(b), "l"(c)); return r; }
__device__ __forceinline__ pk2 add2(pk2 a, pk2 b) { pk2 r; asm("add.rn.f32x2 %0, %1, %2;" : "=l"(r) : "l"(a), "l"(b)); return r; }
__device__ __forceinline__ pk2 sub2(pk2 a, pk2 b) { pk2 r; asm("sub.rn.f32x2 %0, %1, %2;" : "=l"(r) : "l"(a), "l"(b)); return r; }
__device__ __forceinline__ pk2 mul2(pk2 a, pk2 b) { pk2 r; asm("mul.rn.f32x2 %0, %1, %2;" : "=l"(r) : "l"(a), "l"(b)); return r; }

// a * b:  (a.x b.x, a.y b.x) + (-a.y b.y, a.x b.y)
__device__ __forceinline__ float2 cmul(float2 a, float2 b) {
  return unpk(fma2(pk(b.y, b.y), pk(-a.y, a.x), mul2(pk(b.x, b.x), pk(a))));
}
// Twiddle in broadcast form (w.x, w.x), (w.y, w.y): a * w is then two packed instructions with no
// negation or move left over (the half swap and the sign of -a.y are operand modifiers).
struct tw4 { pk2 xx, yy; };
__device__ __forceinline__ tw4 make_tw4(float2 w) { tw4 t; t.xx = pk(w.x, w.x); t.yy = pk(w.y, w.y); return t; }
__device__ __forceinline__ tw4 make_tw4(float4 w) { tw4 t; t.xx = pk(w.x, w.y); t.yy = pk(w.z, w.w); return t; }   // table entry {x, x, y, y}
__device__ __forceinline__ float2 cmul_tw(float2 a, tw4 w) { return unpk(fma2(pk(-a.y, a.x), w.yy, mul2(w.xx, pk(a)))); }
__device__ __forceinline__ float2 cadd(float2 a, float2 b) { return unpk(add2(pk(a), pk(b))); }
__device__ __forceinline__ float2 csub(float2 a, float2 b) { return unpk(sub2(pk(a), pk(b))); }

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
    return unpk(fma2(pk(-s, s), pk(d.y, d.x), mul2(pk(c, c), pk(d))));
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


// ---------------------------------------------------------------------------------------------------
// Decimation in time, radix 2, FMA form.  Input in bit-reversed order (x[brev<R>(n)] = input n), output
// in natural order (X[k] = x[k]).  A butterfly with a general twiddle w costs 6 FMAs instead of the
// 8 operations of the multiply-then-add form:  t = a + w b  (4 FMA),  u = 2 a - t  (2 FMA); packed as
// fp32x2 that is 3 instructions, and 2 for the trivial twiddles 1 and i.
// NZ < R declares that only inputs n < NZ are non-zero: their bit-reversed positions are the multiples
// of R/NZ, the first log2(R/NZ) stages reduce to copies and are skipped.
// ---------------------------------------------------------------------------------------------------
template <int Q>
__device__ __forceinline__ void bfly_w32(float2& a, float2& b) {
  constexpr int q = Q & 31;
  if constexpr (q == 0) {
    const float2 t = cadd(a, b), u = csub(a, b);
    a = t; b = u;
  } else if constexpr (q == 8) {            // w = i:  t = a + (-b.y, b.x),  u = a + (b.y, -b.x)
    const pk2 t = add2(pk(a), pk(-b.y, b.x)), u = add2(pk(a), pk(b.y, -b.x));
    a = unpk(t); b = unpk(u);
  } else {                                  // t = a + c b + s (-b.y, b.x);  u = 2 a - t
    constexpr float c = (float)cos32(q), s = (float)sin32(q);
    pk2 t = fma2(pk(c, c), pk(b), pk(a));
    t = fma2(pk(-s, s), pk(b.y, b.x), t);
    const float2 tt = unpk(t);
    b = unpk(fma2(pk(2.f, 2.f), pk(a), pk(-tt.x, -tt.y)));
    a = tt;
  }
}

template <int R, int H, int BASE, int M>
struct DitInner {
  __device__ __forceinline__ static void run(float2 (&x)[R]) {
    if constexpr (M < H) {
      bfly_w32<M * (16 / H)>(x[BASE + M], x[BASE + M + H]);    // W_{2H}^M = W_32^{M*16/H}, M < H <= 16: q < 16
      DitInner<R, H, BASE, M + 1>::run(x);
    }
  }
};
template <int R, int H, int BASE>
struct DitBlocks {
  __device__ __forceinline__ static void run(float2 (&x)[R]) {
    if constexpr (BASE < R) {
      DitInner<R, H, BASE, 0>::run(x);
      DitBlocks<R, H, BASE + 2 * H>::run(x);
    }
  }
};
template <int R, int H>
struct DitStages {
  __device__ __forceinline__ static void run(float2 (&x)[R]) {
    if constexpr (H < R) {
      DitBlocks<R, H, 0>::run(x);
      DitStages<R, H * 2>::run(x);
    }
  }
};

template <int R, int NZ = R>
__device__ __forceinline__ void fft_dit(float2 (&x)[R]) {
  static_assert(R >= 1 && R <= 32 && (R & (R - 1)) == 0, "R must be a power of two <= 32");
  static_assert(NZ >= 1 && NZ <= R && (NZ & (NZ - 1)) == 0, "NZ must be a power of two <= R");
  constexpr int REP = R / NZ;                 // only positions that are multiples of REP hold data
  if constexpr (REP > 1) {
#pragma unroll
    for (int i = 0; i < R; ++i)
      if (i % REP != 0) x[i] = x[i - i % REP];
  }
  DitStages<R, REP>::run(x);
}

}  // namespace gwmf
