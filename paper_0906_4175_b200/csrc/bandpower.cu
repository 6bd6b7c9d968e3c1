// bandpower.cu -- decimated path, the chi^2 side of step a3/a4 for the narrow bands (class S: at most s_bins bins).
//
// Eq. 5 needs sum_l |z_l[j]|^2 at every sample j (identity P7: sum_l |z_l - z/p|^2 =
// sum_l |z_l|^2 - |z|^2/p).  A band of B contiguous bins gives z_l[j] = e^{2 pi i j e_l/n} y_l[j] with y_l
// band-limited to B bins, so u_l[j] = |z_l[j]|^2 = |y_l[j]|^2 is a REAL series whose spectrum lives on the bins
// |m| < B:  u_l[j] = sum_{|m|<B} U_l[m] e^{2 pi i jm/n},  U_l[m] = sum_k Q[k+m] conj(Q[k]).  Sampling u_l on a
// coarse grid of L >= 2B points (every (n/L)-th sample) therefore loses nothing:
//     y_l[j'] = sum_{i<B} Q[e_l + i] e^{2 pi i j' i/L}            (L-point inverse transform of the band, in shared memory)
//     w_l[j'] = |y_l[j']|^2 = u_l[j' n/L]
//     U_l[m]  = (1/L) sum_{j'} w_l[j'] e^{-2 pi i j' m/L},  |m| < L/2   (L-point forward transform)
// The spectra of all class-S bands of a template are added bin by bin in a fixed order,
//     U+[m] = (m == 0 ? 1 : 2) sum_{l in S} U_l[m],  0 <= m < u_hi = max_l B_l,
// and ONE n-point inverse transform of U+ (an "effective band" of the two-pass FFT, pass1.cu / pass2.cu) returns
// sum_{l in S} |z_l[j]|^2 = Re IFFT_n(U+)[j] at every sample: exact trigonometric interpolation, no approximation.
// The p n-point transforms of the paper's Fig. 3 become: one for z (the union of the S bands), one
// for U+, one per wide (class D) band -- about 2.7 instead of 16 at the headline config -- plus 2 L-point
// transforms per narrow band, L = 2^11 .. 2^14 (a few percent of one n-point transform each).
//
// The L-point transforms run in place in shared memory as radix 32 x 32 x (L/1024): decimation in frequency on the
// way in (natural -> digit-reversed order), |.|^2 element-wise, decimation in time on the way out (digit-reversed ->
// natural): no permutation pass.  The forward transform of the real w is conj(inverse transform).
#include "fft_reg.cuh"
#include "gwmf_internal.cuh"

namespace gwmf {

__device__ __forceinline__ int pad16(int i) { return i + (i >> 4); }        // one float2 of padding per 16: the
                                                                            // stride-1 groups of the last stage become conflict-free
constexpr int kBpThreads = 256;
constexpr int kTwLo = 128;            // e^{2 pi i t/L} = TWH[t >> 7] * TWL[t & 127]: two small shared tables instead of one
                                      // scattered 8-byte global load per twiddle (every lane in its own sector)
constexpr size_t bp_smem(int log_l) {
  return (size_t)((1 << log_l) + ((1 << log_l) >> 4) + kTwLo + ((1 << log_l) / kTwLo)) * sizeof(float2);
}

template <int LOG_L>
struct BpTw {
  const float2* hi;                   // [L / 128]  e^{2 pi i 128 t/L}
  const float2* lo;                   // [128]      e^{2 pi i t/L}
  __device__ __forceinline__ float2 operator()(int t) const {      // t already reduced mod L
    return cmul(hi[t >> 7], lo[t & (kTwLo - 1)]);
  }
};

// grid (p, templates of the batch), one kernel per coarse-grid size L = 2^LOG_L (a CTA whose band wants another size
// exits at once): W[tb][l][m] = one-sided power spectrum of class-S band l, 0 <= m < B_l.
template <int LOG_L>
__global__ void __launch_bounds__(kBpThreads, LOG_L == 14 ? 1 : 2)
    k_bandpower(const TemplateMeta* __restrict__ meta, const float2* __restrict__ q, const float2* __restrict__ tw_l,
                float2* __restrict__ wbuf, int p, int half_n) {
  constexpr int L = 1 << LOG_L;
  constexpr int R3 = L / 1024;                    // last radix: 2, 4, 8, 16
  constexpr int S1 = L / 32;                      // stride of the first radix-32 stage
  constexpr int TWS = kLMax / L;                  // tw_l[t * TWS] = e^{2 pi i t / L}
  extern __shared__ __align__(16) float2 sm[];
  const int l = blockIdx.x, tb = blockIdx.y;
  const TemplateMeta* mt = meta + tb;
  if (!((mt->s_mask >> l) & 1u)) return;
  const int e_lo = mt->edges[l], B = mt->edges[l + 1] - e_lo;
  int log_l = kLogLMin;
  while ((1 << log_l) < 2 * B) ++log_l;
  if (log_l != LOG_L) return;
  float2* __restrict__ wout = wbuf + ((size_t)tb * p + l) * kUCap;
  const int tid = threadIdx.x;
  float2* twl = sm + L + (L >> 4);
  float2* twh = twl + kTwLo;
  for (int i = tid; i < kTwLo; i += kBpThreads) twl[i] = tw_l[i * TWS];
  for (int i = tid; i < L / kTwLo; i += kBpThreads) twh[i] = tw_l[i * kTwLo * TWS];
  BpTw<LOG_L> tw;
  tw.hi = twh;
  tw.lo = twl;

  // the band's bins -> shared memory.  Q is stored c-major inside each row of 1024 bins (cm_pos): walk the band's rows
  // position by position (coalesced) and scatter to the bin's place
  for (int i = B + tid; i < L; i += kBpThreads) sm[pad16(i)] = make_float2(0.f, 0.f);
  {
    const int row_lo = e_lo >> kLogN2, n_rows = ((e_lo + B - 1) >> kLogN2) - row_lo + 1;
    const float2* __restrict__ qrows = q + (size_t)tb * half_n + (size_t)row_lo * kN2;
    for (int idx = tid; idx < n_rows * kN2; idx += kBpThreads) {
      const int i = ((row_lo + (idx >> kLogN2)) << kLogN2) + cm_pos(idx & (kN2 - 1)) - e_lo;
      if (i >= 0 && i < B) sm[pad16(i)] = qrows[idx];
    }
  }
  __syncthreads();
  // ---- inverse transform, decimation in frequency: stage 1 (inputs i >= L/2 are zero since L >= 2B)
#pragma unroll 1
  for (int o = tid; o < S1; o += kBpThreads) {
    float2 x[32];
#pragma unroll
    for (int qq = 0; qq < 16; ++qq) x[brev<32>(qq)] = sm[pad16(o + S1 * qq)];
    fft_dit<32, 16>(x);
#pragma unroll
    for (int k = 0; k < 32; ++k) sm[pad16(o + S1 * k)] = k == 0 ? x[0] : cmul(x[k], tw((o * k) & (L - 1)));
  }
  __syncthreads();
  // ---- stage 2: inside each block k1 of S1 = 32 R3 points
#pragma unroll 1
  for (int g = tid; g < S1; g += kBpThreads) {
    const int k1 = g / R3, o2 = g - k1 * R3, base = k1 * S1 + o2;
    float2 x[32];
#pragma unroll
    for (int qq = 0; qq < 32; ++qq) x[brev<32>(qq)] = sm[pad16(base + R3 * qq)];
    fft_dit<32>(x);
#pragma unroll
    for (int k = 0; k < 32; ++k) sm[pad16(base + R3 * k)] = k == 0 ? x[0] : cmul(x[k], tw((32 * o2 * k) & (L - 1)));
  }
  __syncthreads();
  // ---- stage 3 (R3 points, stride 1), |y|^2, and the first stage of the way back (same groups, no twiddle)
#pragma unroll 1
  for (int g = tid; g < 1024; g += kBpThreads) {
    const int base = g * R3;
    float2 x[R3];
#pragma unroll
    for (int qq = 0; qq < R3; ++qq) x[brev<R3>(qq)] = sm[pad16(base + qq)];
    fft_dit<R3>(x);
    float2 w[R3];
#pragma unroll
    for (int qq = 0; qq < R3; ++qq) w[brev<R3>(qq)] = make_float2(fmaf(x[qq].x, x[qq].x, x[qq].y * x[qq].y), 0.f);
    fft_dit<R3>(w);
#pragma unroll
    for (int k = 0; k < R3; ++k) sm[pad16(base + k)] = w[k];
  }
  __syncthreads();
  // ---- decimation in time: twiddle first, then the radix-32 transform (transposes of stages 2 and 1)
#pragma unroll 1
  for (int g = tid; g < S1; g += kBpThreads) {
    const int k1 = g / R3, o2 = g - k1 * R3, base = k1 * S1 + o2;
    float2 x[32];
#pragma unroll
    for (int qq = 0; qq < 32; ++qq) {
      const float2 v = sm[pad16(base + R3 * qq)];
      x[brev<32>(qq)] = qq == 0 ? v : cmul(v, tw((32 * o2 * qq) & (L - 1)));
    }
    fft_dit<32>(x);
#pragma unroll
    for (int k = 0; k < 32; ++k) sm[pad16(base + R3 * k)] = x[k];
  }
  __syncthreads();
  // last stage: only the outputs m = o + S1 k < B <= L/2 are wanted, i.e. k < 16; they leave straight to global memory
  const float inv_l = 1.0f / (float)L;
#pragma unroll 1
  for (int o = tid; o < S1; o += kBpThreads) {
    float2 x[32];
#pragma unroll
    for (int qq = 0; qq < 32; ++qq) {
      const float2 v = sm[pad16(o + S1 * qq)];
      x[brev<32>(qq)] = qq == 0 ? v : cmul(v, tw((o * qq) & (L - 1)));
    }
    fft_dit<32>(x);
#pragma unroll
    for (int k = 0; k < 16; ++k) {
      const int m = o + S1 * k;
      if (m < B) {
        const float sc = m == 0 ? inv_l : 2.0f * inv_l;                  // one-sided: U+[m] = 2 U[m] for m > 0
        wout[m] = make_float2(x[k].x * sc, -x[k].y * sc);               // conj: forward transform of a real series
      }
    }
  }
}

// U+[tb][m] = sum over the class-S bands, ascending l (fixed order: bit-reproducible), 0 <= m < u_hi
__device__ __forceinline__ float2 usum(const TemplateMeta* mt, const float2* __restrict__ wbuf, int tb, int p, int m) {
  float2 acc = make_float2(0.f, 0.f);
  unsigned s = mt->s_mask;
  while (s) {
    const int l = __ffs(s) - 1;
    s &= s - 1;
    if (m < mt->edges[l + 1] - mt->edges[l]) {
      const float2 v = wbuf[((size_t)tb * p + l) * kUCap + m];
      acc.x += v.x;
      acc.y += v.y;
    }
  }
  return acc;
}

// Unpaired template: ubuf[tb][m] = U+[m] (one-sided, doubled for m > 0: its transform's real part is u).
// Owner of a pair (tb, tb + 1): the two ubuf rows hold the pair spectrum P[m] = U_A[m] + i U_B[m], -up_hi < m < up_hi,
// with bin 0 at the start of the guest's row; U_X[m] = U+_X[m] / 2 for m > 0, U_X[-m] = conj(U_X[m]) (two-sided
// spectrum of a real series), so that ONE transform returns u_A + i u_B.
__global__ void __launch_bounds__(256) k_uspec(const TemplateMeta* __restrict__ meta, const float2* __restrict__ wbuf,
                                               float2* __restrict__ ubuf, int p) {
  const int tb = blockIdx.y, m = blockIdx.x * 256 + threadIdx.x;
  const TemplateMeta* mt = meta + tb;
  if (mt->pair == 2 || !mt->s_mask) return;               // a guest's spectrum is written by its owner
  // rows of 1024 bins are stored c-major (cm_pos), as pass 1 reads them; bin -m sits in row floor(-m / 1024)
  const int mp = (m & ~(kN2 - 1)) + cm_pos(m & (kN2 - 1));
  if (mt->pair == 0) {
    if (m < mt->u_hi) ubuf[(size_t)tb * kUCap + mp] = usum(mt, wbuf, tb, p, m);
    return;
  }
  if (m >= mt->up_hi) return;
  const float2 ua = usum(mt, wbuf, tb, p, m), ub = usum(mt + 1, wbuf, tb + 1, p, m);
  float2* bin0 = ubuf + (size_t)(tb + 1) * kUCap;
  if (m == 0) {
    bin0[0] = make_float2(ua.x, ub.x);                    // both are real at m = 0
  } else {
    const int km = -m, kmp = (km & ~(kN2 - 1)) + cm_pos(km & (kN2 - 1));        // (km & ~1023) = 1024 floor(km / 1024) < 0
    bin0[mp] = make_float2(0.5f * (ua.x - ub.y), 0.5f * (ua.y + ub.x));        // (U_A + i U_B) / 2
    bin0[kmp] = make_float2(0.5f * (ua.x + ub.y), 0.5f * (ub.x - ua.y));       // (conj U_A + i conj U_B) / 2
  }
}

cudaError_t configure_bandpower() {
  cudaError_t e = cudaFuncSetAttribute(k_bandpower<11>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)bp_smem(11));
  if (e == cudaSuccess) e = cudaFuncSetAttribute(k_bandpower<12>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)bp_smem(12));
  if (e == cudaSuccess) e = cudaFuncSetAttribute(k_bandpower<13>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)bp_smem(13));
  if (e == cudaSuccess) e = cudaFuncSetAttribute(k_bandpower<14>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)bp_smem(14));
  return e;
}

cudaError_t launch_bandpower(Ctx* c, int first, int count, int parity, cudaStream_t st) {
  const int p = c->prm.p;
  const size_t half = (size_t)(c->n / 2);
  const TemplateMeta* meta = ws_ptr<TemplateMeta>(c, c->lay.meta) + first;
  const float2* q = ws_ptr<float2>(c, c->lay.q) + (size_t)parity * c->lay.batch * half;
  float2* wbuf = ws_ptr<float2>(c, c->lay.wbuf) + (size_t)parity * c->lay.batch * p * kUCap;
  float2* ubuf = ws_ptr<float2>(c, c->lay.ubuf) + (size_t)parity * c->lay.batch * kUCap;
  const float2* tw_l = ws_ptr<float2>(c, c->lay.tw_l);
  const dim3 grid(p, count);
  // one launch per coarse-grid size that the class threshold allows (a band of B bins uses L = 2^ceil(log2 2B) >= 2048)
  k_bandpower<11><<<grid, kBpThreads, bp_smem(11), st>>>(meta, q, tw_l, wbuf, p, (int)half);
  c->launches++;
  if (c->s_bins > 1024) { k_bandpower<12><<<grid, kBpThreads, bp_smem(12), st>>>(meta, q, tw_l, wbuf, p, (int)half); c->launches++; }
  if (c->s_bins > 2048) { k_bandpower<13><<<grid, kBpThreads, bp_smem(13), st>>>(meta, q, tw_l, wbuf, p, (int)half); c->launches++; }
  if (c->s_bins > 4096) { k_bandpower<14><<<grid, kBpThreads, bp_smem(14), st>>>(meta, q, tw_l, wbuf, p, (int)half); c->launches++; }
  k_uspec<<<dim3(c->s_bins / 256, count), 256, 0, st>>>(meta, wbuf, ubuf, p);
  c->launches++;
  return cudaGetLastError();
}

}  // namespace gwmf
