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

// threads per CTA = work items of a radix-32 stage (L / 32), so that every thread has one: 128 for L <= 4096 (4 CTAs per
// SM), 256 for L = 8192 (2 per SM), 512 for L = 16384 (1 per SM: 140 KB of shared memory)
constexpr int bp_threads(int log_l) { return log_l <= 12 ? 128 : log_l == 13 ? 256 : 512; }
constexpr int bp_ctas(int log_l) { return log_l <= 12 ? 4 : log_l == 13 ? 2 : 1; }
constexpr int kTwLo = 128;            // e^{2 pi i t/L} = TWH[t >> 7] * TWL[t & 127]: two small shared tables instead of one
                                      // scattered 8-byte global load per twiddle (every lane in its own sector)
constexpr size_t bp_smem(int log_l) {
  return (size_t)((1 << log_l) + ((1 << log_l) >> 4) + ((1 << log_l) >> 5) + kTwLo + ((1 << log_l) / kTwLo)) * sizeof(float2);
}

template <int LOG_L>
struct BpTw {
  const float2* hi;                   // [L / 128]  e^{2 pi i 128 t/L}
  const float2* lo;                   // [128]      e^{2 pi i t/L}
  __device__ __forceinline__ float2 operator()(int t) const {      // t already reduced mod L
    return cmul(hi[t >> 7], lo[t & (kTwLo - 1)]);
  }
};

// The 32 twiddles e^{2 pi i step k/L}, k = 0..31, of one work item of a radix-32 stage: a geometric sequence.  Two table
// look-ups (w = e^{2 pi i step/L} and w^8, both exact to one rounding) and short products: w^(8a + b) = (w^8)^a w^b, at
// most 3 + 7 multiplications deep, instead of 31 look-ups (the shared-memory pipe is these kernels' busiest unit).
template <int LOG_L>
struct BpSeq {
  float2 lo[8];      // w^b
  float2 hi[4];      // w^(8a)
  __device__ __forceinline__ BpSeq(const BpTw<LOG_L>& tw, int step) {
    constexpr int L = 1 << LOG_L;
    const float2 w1 = tw(step & (L - 1)), w8 = tw((8 * step) & (L - 1));
    lo[0] = make_float2(1.f, 0.f);
    lo[1] = w1;
#pragma unroll
    for (int b = 2; b < 8; ++b) lo[b] = cmul(lo[b - 1], w1);
    hi[0] = make_float2(1.f, 0.f);
    hi[1] = w8;
    hi[2] = cmul(w8, w8);
    hi[3] = cmul(hi[2], w8);
  }
  __device__ __forceinline__ float2 mul(float2 v, int k) const {      // v e^{2 pi i step k/L}, k a compile-time constant after unrolling
    const int a = k >> 3, b = k & 7;
    if (k == 0) return v;
    if (a == 0) return cmul(v, lo[b]);
    if (b == 0) return cmul(v, hi[a]);
    return cmul(cmul(v, lo[b]), hi[a]);
  }
};

// Job lists of a batch, one per kernel: class 0..3 = bands on a grid of 2^11..2^14 points, class 4 = the sub-grid jobs
// (band, r) of the bands on 2^15 / 2^16 points.  jobs[class][i] = tb << 16 | l << 8 | r.  The order inside a list is
// whatever the atomics give: every job writes rows of its own, so the results do not depend on it.
constexpr int kBpJobCap = kMaxBatch * kMaxBands * kSubMax;
constexpr int kBpClasses = 5;
__global__ void __launch_bounds__(1024) k_bp_jobs(const TemplateMeta* __restrict__ meta, int p, int count, int* __restrict__ jobs,
                                                  int* __restrict__ n_jobs) {
  __shared__ int s_n[kBpClasses];
  if (threadIdx.x < kBpClasses) s_n[threadIdx.x] = 0;
  __syncthreads();
  for (int i = threadIdx.x; i < count * p; i += blockDim.x) {
    const int tb = i / p, l = i - tb * p;
    const TemplateMeta* mt = meta + tb;
    if (!((mt->s_mask >> l) & 1u)) continue;
    const int B = mt->edges[l + 1] - mt->edges[l];
    int log_l = kLogLMin;
    while ((1 << log_l) < 2 * B) ++log_l;
    if (log_l <= 14) {
      jobs[(log_l - kLogLMin) * kBpJobCap + atomicAdd(&s_n[log_l - kLogLMin], 1)] = (tb << 16) | (l << 8);
    } else {
      const int sub = 1 << (log_l - 14);
      const int at = atomicAdd(&s_n[4], sub);
      for (int r = 0; r < sub; ++r) jobs[4 * kBpJobCap + at + r] = (tb << 16) | (l << 8) | r;
    }
  }
  __syncthreads();
  if (threadIdx.x < kBpClasses) n_jobs[threadIdx.x] = s_n[threadIdx.x];
}

// grid (p, templates of the batch), one kernel per coarse-grid size L = 2^LOG_L (a CTA whose band wants another size
// exits at once): W[tb][l][m] = one-sided power spectrum of class-S band l, 0 <= m < B_l.
// The CTAs of a launch walk over the job list of their class (k_bp_jobs): only CTAs with work are started.
// SUB (LOG_L = 14 only): the band needs a grid of LT = 2^15 or 2^16 points.  CTA r = blockIdx.z < D = LT / L takes the
// interleaved sub-grid j' = r + D j'':
//     y[r + D j''] = sum_{i' < L} X_r[i'] e^{2 pi i j'' i'/L},   X_r[i'] = sum_q Q[e_l + i' + q L] e^{2 pi i r (i' + q L)/LT}
// (the band's bins with the sub-grid's phase ramp, folded modulo L), and its share of the LT-point forward transform,
//     U_l[m] += (1/LT) e^{-2 pi i r m/LT} W_r[m mod L],   W_r = L-point forward transform of |y[r + D j'']|^2,
// goes to row r of the band's rows of wbuf; k_uspec adds the rows in a fixed order.
template <int LOG_L, bool SUB>
__global__ void __launch_bounds__(bp_threads(LOG_L), bp_ctas(LOG_L))
    k_bandpower(const TemplateMeta* __restrict__ meta, const float2* __restrict__ q, const float2* __restrict__ tw_l,
                float2* __restrict__ wbuf, int p, int half_n, const int* __restrict__ jobs, const int* __restrict__ n_jobs) {
  constexpr int L = 1 << LOG_L;
  constexpr int NT = bp_threads(LOG_L);
  constexpr int R3 = L / 1024;                    // last radix: 2, 4, 8, 16
  constexpr int S1 = L / 32;                      // stride of the first radix-32 stage
  constexpr int TWS = kLMax / L;                  // tw_l[t * TWS] = e^{2 pi i t / L}
  constexpr int CLS = SUB ? 4 : LOG_L - kLogLMin; // job class (k_bp_jobs)
  extern __shared__ __align__(16) float2 sm[];
  // element i of the L-point array: one float2 of padding per 16 (the stride-1 groups of the last radix become
  // conflict-free) and R3 more per block of S1 = L / 32 (so do the stride-R3 accesses of the middle radix-32 stage, whose
  // lanes sit in different blocks)
  auto pd = [](int i) { return i + (i >> 4) + (i >> (LOG_L - 5)) * R3; };
  __shared__ float2 s_fine[4];
  const int n_job = n_jobs[CLS];
  if ((int)blockIdx.x >= n_job) return;
  const int tid = threadIdx.x;
  float2* twl = sm + L + (L >> 4) + (L >> 5);
  float2* twh = twl + kTwLo;
  for (int i = tid; i < kTwLo; i += NT) twl[i] = tw_l[i * TWS];
  for (int i = tid; i < L / kTwLo; i += NT) twh[i] = tw_l[i * kTwLo * TWS];
  BpTw<LOG_L> tw;
  tw.hi = twh;
  tw.lo = twl;

#pragma unroll 1
  for (int job = blockIdx.x; job < n_job; job += gridDim.x) {
  const int jd = jobs[CLS * kBpJobCap + job];     // tb << 16 | l << 8 | sub-grid r
  const int tb = jd >> 16, l = (jd >> 8) & 255, r = jd & 255;
  const TemplateMeta* mt = meta + tb;
  const int e_lo = mt->edges[l], B = mt->edges[l + 1] - e_lo;
  int log_lt = kLogLMin;                          // the band's whole grid LT = 2^log_lt (= L unless SUB)
  while ((1 << log_lt) < 2 * B) ++log_lt;
  float2* __restrict__ wout = wbuf + (((size_t)tb * p + l) * kSubMax + r) * kUCap;
  __syncthreads();                                // the previous job of this CTA is done with shared memory; tables are in place

  // e^{2 pi i t/LT}, LT = 2^15 or 2^16 (SUB): t = (t >> sh) on the L-point table times the few finer steps below it
  const int sh = log_lt - LOG_L;                  // 1 or 2
  if constexpr (SUB) {
    if (tid < 4) {
      float sn, cs;
      sincospif(2.0f * (float)tid / (float)(1u << log_lt), &sn, &cs);
      s_fine[tid] = make_float2(cs, sn);
    }
    __syncthreads();                              // twl / twh / s_fine are in place
  }
  auto sub_tw = [&](unsigned t) -> float2 {
    t &= (1u << log_lt) - 1u;
    const float2 coarse = tw((int)(t >> sh));
    const unsigned lo = t & ((1u << sh) - 1u);
    return lo ? cmul(coarse, s_fine[lo]) : coarse;
  };
  // the band's bins -> shared memory.  Q is stored c-major inside each row of 1024 bins (cm_pos): walk the band's rows
  // position by position (coalesced) and scatter to the bin's place
  {
    const int row_lo = e_lo >> kLogN2, n_rows = ((e_lo + B - 1) >> kLogN2) - row_lo + 1;
    const float2* __restrict__ qrows = q + (size_t)tb * half_n + (size_t)row_lo * kN2;
    if constexpr (!SUB) {
      for (int i = B + tid; i < L; i += NT) sm[pd(i)] = make_float2(0.f, 0.f);
      for (int idx = tid; idx < n_rows * kN2; idx += NT) {
        const int i = ((row_lo + (idx >> kLogN2)) << kLogN2) + cm_pos(idx & (kN2 - 1)) - e_lo;
        if (i >= 0 && i < B) sm[pd(i)] = qrows[idx];
      }
    } else {
      // X_r[i mod L] += Q[e_l + i] e^{2 pi i r i/LT}: a cell receives at most two terms (B <= LT / 2 = 2 L), so the
      // shared-memory adds commute and the result does not depend on their order
      for (int i = tid; i < L; i += NT) sm[pd(i)] = make_float2(0.f, 0.f);
      __syncthreads();
      for (int idx0 = tid; idx0 < n_rows * kN2; idx0 += 4 * NT) {
        float2 v[4];
        int ii[4];
#pragma unroll
        for (int u = 0; u < 4; ++u) {                                      // four loads in flight
          const int idx = idx0 + u * NT;
          ii[u] = ((row_lo + (idx >> kLogN2)) << kLogN2) + cm_pos(idx & (kN2 - 1)) - e_lo;
          if (idx >= n_rows * kN2 || ii[u] >= B) ii[u] = -1;
          v[u] = ii[u] >= 0 ? __ldg(qrows + idx) : make_float2(0.f, 0.f);
        }
#pragma unroll
        for (int u = 0; u < 4; ++u) {
          if (ii[u] < 0) continue;
          const float2 t = r ? cmul(v[u], sub_tw((unsigned)r * (unsigned)ii[u])) : v[u];
          float* dst = reinterpret_cast<float*>(&sm[pd(ii[u] & (L - 1))]);
          atomicAdd(dst, t.x);
          atomicAdd(dst + 1, t.y);
        }
      }
    }
  }
  __syncthreads();
  // ---- inverse transform, decimation in frequency: stage 1 (!SUB: inputs i >= L/2 are zero since L >= 2B)
#pragma unroll 1
  for (int o = tid; o < S1; o += NT) {
    float2 x[32];
#pragma unroll
    if constexpr (!SUB) {
#pragma unroll
      for (int qq = 0; qq < 16; ++qq) x[brev<32>(qq)] = sm[pd(o + S1 * qq)];
      fft_dit<32, 16>(x);
    } else {                                      // a folded band fills the whole sub-grid spectrum
#pragma unroll
      for (int qq = 0; qq < 32; ++qq) x[brev<32>(qq)] = sm[pd(o + S1 * qq)];
      fft_dit<32>(x);
    }
#pragma unroll
    const BpSeq<LOG_L> sq(tw, o);
#pragma unroll
    for (int k = 0; k < 32; ++k) sm[pd(o + S1 * k)] = sq.mul(x[k], k);
  }
  __syncthreads();
  // ---- stage 2: inside each block k1 of S1 = 32 R3 points
#pragma unroll 1
  for (int g = tid; g < S1; g += NT) {
    const int k1 = g / R3, o2 = g - k1 * R3, base = k1 * S1 + o2;
    float2 x[32];
#pragma unroll
    for (int qq = 0; qq < 32; ++qq) x[brev<32>(qq)] = sm[pd(base + R3 * qq)];
    fft_dit<32>(x);
#pragma unroll
    const BpSeq<LOG_L> sq(tw, 32 * o2);
#pragma unroll
    for (int k = 0; k < 32; ++k) sm[pd(base + R3 * k)] = sq.mul(x[k], k);
  }
  __syncthreads();
  // ---- stage 3 (R3 points, stride 1), |y|^2, and the first stage of the way back (same groups, no twiddle)
#pragma unroll 1
  for (int g = tid; g < 1024; g += NT) {
    const int base = g * R3;
    float2 x[R3];
#pragma unroll
    for (int qq = 0; qq < R3; ++qq) x[brev<R3>(qq)] = sm[pd(base + qq)];
    fft_dit<R3>(x);
    float2 w[R3];
#pragma unroll
    for (int qq = 0; qq < R3; ++qq) w[brev<R3>(qq)] = make_float2(fmaf(x[qq].x, x[qq].x, x[qq].y * x[qq].y), 0.f);
    fft_dit<R3>(w);
#pragma unroll
    for (int k = 0; k < R3; ++k) sm[pd(base + k)] = w[k];
  }
  __syncthreads();
  // ---- decimation in time: twiddle first, then the radix-32 transform (transposes of stages 2 and 1)
#pragma unroll 1
  for (int g = tid; g < S1; g += NT) {
    const int k1 = g / R3, o2 = g - k1 * R3, base = k1 * S1 + o2;
    const BpSeq<LOG_L> sq(tw, 32 * o2);
    float2 x[32];
#pragma unroll
    for (int qq = 0; qq < 32; ++qq) {
      const float2 v = sm[pd(base + R3 * qq)];
      x[brev<32>(qq)] = sq.mul(v, qq);
    }
    fft_dit<32>(x);
#pragma unroll
    for (int k = 0; k < 32; ++k) sm[pd(base + R3 * k)] = x[k];
  }
  __syncthreads();
  // last stage: only the outputs m = o + S1 k < B <= L/2 are wanted, i.e. k < 16; they leave straight to global memory
  const float inv_l = 1.0f / (float)(1u << log_lt);
#pragma unroll 1
  for (int o = tid; o < S1; o += NT) {
    const BpSeq<LOG_L> sq(tw, o);
    float2 x[32];
#pragma unroll
    for (int qq = 0; qq < 32; ++qq) {
      const float2 v = sm[pd(o + S1 * qq)];
      x[brev<32>(qq)] = sq.mul(v, qq);
    }
    fft_dit<32>(x);
    if constexpr (!SUB) {
#pragma unroll
      for (int k = 0; k < 16; ++k) {
        const int m = o + S1 * k;
        if (m < B) {
          const float sc = m == 0 ? inv_l : 2.0f * inv_l;                  // one-sided: U+[m] = 2 U[m] for m > 0
          wout[m] = make_float2(x[k].x * sc, -x[k].y * sc);               // conj: forward transform of a real series
        }
      }
    } else {
      // W_r is periodic in m with period L: every m = m' + fold L < B gets conj(x) e^{-2 pi i r m/LT}
#pragma unroll
      for (int k = 0; k < 32; ++k) {
        const float2 wc = make_float2(x[k].x, -x[k].y);                    // conj: forward transform of a real series
        for (int m = o + S1 * k; m < B; m += L) {
          const float sc = m == 0 ? inv_l : 2.0f * inv_l;                  // one-sided: U+[m] = 2 U[m] for m > 0
          const float2 t = sub_tw((unsigned)r * (unsigned)m);
          const float2 v = r ? cmul(wc, make_float2(t.x, -t.y)) : wc;      // e^{-2 pi i r m/LT}
          wout[m] = make_float2(v.x * sc, v.y * sc);
        }
      }
    }
  }
  }   // job
}

// U+[tb][m] = sum over the rows of wbuf of the class-S bands, ascending (l, sub-grid): a fixed order, bit-reproducible.
// The rows in use and their lengths are listed in shared memory once per CTA.
constexpr int kUsEntries = kMaxBands * kSubMax;
// called by one whole warp (lane = band)
__device__ __forceinline__ void uspec_list(const TemplateMeta* mt, int tb, int p, int* s_row, int* s_len, int* s_n) {
  const int l = threadIdx.x & 31;
  const bool is_s = (mt->s_mask >> l) & 1u;
  const int B = is_s ? mt->edges[l + 1] - mt->edges[l] : 0;
  const int sub = !is_s ? 0 : B > kLMax ? 4 : B > kLMax / 2 ? 2 : 1;      // grid 2^16, 2^15, <= 2^14: rows of wbuf in use
  int incl = sub;
#pragma unroll
  for (int d = 1; d < 32; d <<= 1) {
    const int v = __shfl_up_sync(0xFFFFFFFFu, incl, d);
    if (l >= d) incl += v;
  }
  for (int r = 0; r < sub; ++r) { s_row[incl - sub + r] = (tb * p + l) * kSubMax + r; s_len[incl - sub + r] = B; }
  if (l == 31) *s_n = incl;
}
__device__ __forceinline__ void uspec_sum(const float2* __restrict__ wbuf, const int* s_row, const int* s_len, int n, int m0,
                                          float2 (&acc)[4]) {
#pragma unroll
  for (int i = 0; i < 4; ++i) acc[i] = make_float2(0.f, 0.f);
  for (int e = 0; e < n; ++e) {
    const float2* __restrict__ row = wbuf + (size_t)s_row[e] * kUCap;
    const int B = s_len[e];
#pragma unroll
    for (int i = 0; i < 4; ++i) {
      const int m = m0 + 256 * i;
      if (m < B) {
        const float2 v = __ldg(row + m);
        acc[i].x += v.x;
        acc[i].y += v.y;
      }
    }
  }
}

// Unpaired template: ubuf[tb][m] = U+[m] (one-sided, doubled for m > 0: its transform's real part is u).
// Owner of a pair (tb, tb + 1): the two ubuf rows hold the pair spectrum P[m] = U_A[m] + i U_B[m], -up_hi < m < up_hi,
// with bin 0 at the start of the guest's row; U_X[m] = U+_X[m] / 2 for m > 0, U_X[-m] = conj(U_X[m]) (two-sided
// spectrum of a real series), so that ONE transform returns u_A + i u_B.
// A CTA owns the 1024 bins m = 1024 b .. 1024 b + 1023 of one template (pair); the rows of 1024 bins are stored
// c-major (cm_pos), as pass 1 reads them, so the results are transposed through shared memory and leave coalesced.
// Bin -m sits in row floor(-m / 1024): row -b for m = 1024 b, row -b - 1 for the other 1023.
__global__ void __launch_bounds__(256) k_uspec(const TemplateMeta* __restrict__ meta, const float2* __restrict__ wbuf,
                                               float2* __restrict__ ubuf, int p) {
  __shared__ int s_row[2][kUsEntries], s_len[2][kUsEntries], s_n[2];
  __shared__ float2 s_pos[kN2 + 32], s_neg[kN2 + 32];
  const int tb = blockIdx.y, b = blockIdx.x, tid = threadIdx.x;
  const TemplateMeta* mt = meta + tb;
  const int pair = mt->pair;
  if (pair == 2 || !mt->s_mask) return;                   // a guest's spectrum is written by its owner
  const int hi = pair ? mt->up_hi : mt->u_hi;
  if (b * kN2 >= hi) return;
  if (tid < 32) uspec_list(mt, tb, p, s_row[0], s_len[0], &s_n[0]);
  else if (tid < 64 && pair) uspec_list(mt + 1, tb + 1, p, s_row[1], s_len[1], &s_n[1]);
  __syncthreads();
  const int m0 = b * kN2 + tid;
  float2 ua[4], ub[4];
  uspec_sum(wbuf, s_row[0], s_len[0], s_n[0], m0, ua);
  if (pair) uspec_sum(wbuf, s_row[1], s_len[1], s_n[1], m0, ub);
#pragma unroll
  for (int i = 0; i < 4; ++i) {
    const int k2 = tid + 256 * i, pp = cm_pos(k2);
    if (!pair) {
      s_pos[pp + (pp >> 5)] = ua[i];
    } else {
      const int kn = (kN2 - k2) & (kN2 - 1), pn = cm_pos(kn);              // bin -m has k2' = (-m) mod 1024
      float2 vp, vn;
      if (m0 + 256 * i == 0) {
        vp = vn = make_float2(ua[i].x, ub[i].x);                          // both are real at m = 0
      } else {
        vp = make_float2(0.5f * (ua[i].x - ub[i].y), 0.5f * (ua[i].y + ub[i].x));        // (U_A + i U_B) / 2
        vn = make_float2(0.5f * (ua[i].x + ub[i].y), 0.5f * (ub[i].x - ua[i].y));        // (conj U_A + i conj U_B) / 2
      }
      s_pos[pp + (pp >> 5)] = vp;
      s_neg[pn + (pn >> 5)] = vn;
    }
  }
  __syncthreads();
  float2* bin0 = ubuf + (size_t)(pair ? tb + 1 : tb) * kUCap;
#pragma unroll
  for (int i = 0; i < 4; ++i) {
    const int pos = tid + 256 * i, k2 = cm_pos(pos);
    if (b * kN2 + k2 < hi) bin0[b * kN2 + pos] = s_pos[pos + (pos >> 5)];
    if (pair) {
      // k2' = k2: bin -(1024 b + 1024 - k2) for k2 >= 1 (row -b - 1); k2' = 0 is bin -1024 b (row -b; bin 0 itself for b = 0)
      const int m = k2 ? (b + 1) * kN2 - k2 : b * kN2;
      if (m < hi && m > 0) bin0[-(k2 ? b + 1 : b) * kN2 + pos] = s_neg[pos + (pos >> 5)];
    }
  }
}

size_t bp_jobs_bytes() { return 2 * (size_t)(kBpClasses * kBpJobCap + 8) * sizeof(int); }

cudaError_t configure_bandpower() {
  cudaError_t e = cudaFuncSetAttribute(k_bandpower<11, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)bp_smem(11));
  if (e == cudaSuccess) e = cudaFuncSetAttribute(k_bandpower<12, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)bp_smem(12));
  if (e == cudaSuccess) e = cudaFuncSetAttribute(k_bandpower<13, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)bp_smem(13));
  if (e == cudaSuccess) e = cudaFuncSetAttribute(k_bandpower<14, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)bp_smem(14));
  if (e == cudaSuccess) e = cudaFuncSetAttribute(k_bandpower<14, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)bp_smem(14));
  return e;
}

cudaError_t launch_bandpower(Ctx* c, int first, int count, int parity, cudaStream_t st) {
  const int p = c->prm.p;
  const size_t half = (size_t)(c->n / 2);
  const TemplateMeta* meta = ws_ptr<TemplateMeta>(c, c->lay.meta) + first;
  const float2* q = ws_ptr<float2>(c, c->lay.q) + (size_t)parity * c->lay.batch * half;
  float2* wbuf = ws_ptr<float2>(c, c->lay.wbuf) + (size_t)parity * c->lay.batch * p * kSubMax * kUCap;
  float2* ubuf = ws_ptr<float2>(c, c->lay.ubuf) + (size_t)parity * c->lay.batch * kUCap;
  const float2* tw_l = ws_ptr<float2>(c, c->lay.tw_l);
  // job lists of the batch (one per kernel), then one launch per coarse-grid size that the class threshold allows (a band
  // of B bins uses L = 2^ceil(log2 2B) >= 2048).  The kernels are independent and each fills only part of the device, so
  // they run side by side: the larger grids on streams of their own between a fork and a join on st.
  int* jobs = ws_ptr<int>(c, c->lay.bp_jobs) + (size_t)parity * (kBpClasses * kBpJobCap + 8);
  int* n_jobs = jobs + kBpClasses * kBpJobCap;
  k_bp_jobs<<<1, 1024, 0, st>>>(meta, p, count, jobs, n_jobs);
  c->launches++;
  cudaError_t e = cudaGetLastError();
  if (e != cudaSuccess) return e;
  const bool fork = c->s_bins > 1024;
  if (fork && (e = cudaEventRecord(c->ev_bp_fork, st)) != cudaSuccess) return e;
  auto grid_of = [&](int log_l) { return bp_ctas(log_l) * c->n_sms; };    // the CTAs of a kernel that can be resident
  k_bandpower<11, false><<<grid_of(11), bp_threads(11), bp_smem(11), st>>>(meta, q, tw_l, wbuf, p, (int)half, jobs, n_jobs);
  c->launches++;
  if ((e = cudaGetLastError()) != cudaSuccess) return e;
  // A side stream must have waited for the fork (the job list of THIS batch) before anything is launched on it: a
  // failed wait is returned, not launched past.
  int used = 0;
  auto side = [&](int i, cudaStream_t* out) -> cudaError_t {
    const cudaError_t w = cudaStreamWaitEvent(c->bp[i], c->ev_bp_fork, 0);
    if (w != cudaSuccess) return w;
    used |= 1 << i;
    *out = c->bp[i];
    return cudaSuccess;
  };
  cudaStream_t sx = nullptr;
  if (c->s_bins > 1024) {
    if ((e = side(0, &sx)) != cudaSuccess) return e;
    k_bandpower<12, false><<<grid_of(12), bp_threads(12), bp_smem(12), sx>>>(meta, q, tw_l, wbuf, p, (int)half, jobs, n_jobs);
    c->launches++;
    if ((e = cudaGetLastError()) != cudaSuccess) return e;
  }
  if (c->s_bins > 2048) {
    if ((e = side(1, &sx)) != cudaSuccess) return e;
    k_bandpower<13, false><<<grid_of(13), bp_threads(13), bp_smem(13), sx>>>(meta, q, tw_l, wbuf, p, (int)half, jobs, n_jobs);
    c->launches++;
    if ((e = cudaGetLastError()) != cudaSuccess) return e;
  }
  if (c->s_bins > 4096) {
    if ((e = side(2, &sx)) != cudaSuccess) return e;
    k_bandpower<14, false><<<grid_of(14), bp_threads(14), bp_smem(14), sx>>>(meta, q, tw_l, wbuf, p, (int)half, jobs, n_jobs);
    c->launches++;
    if ((e = cudaGetLastError()) != cudaSuccess) return e;
  }
  if (c->s_bins > kLMax / 2) {                    // bands on grids of 2^15 or 2^16 points: up to kSubMax sub-grid jobs each
    k_bandpower<14, true><<<grid_of(14), bp_threads(14), bp_smem(14), st>>>(meta, q, tw_l, wbuf, p, (int)half, jobs, n_jobs);
    c->launches++;
    if ((e = cudaGetLastError()) != cudaSuccess) return e;
  }
  for (int i = 0; i < 3; ++i) {
    if (!(used & (1 << i))) continue;
    if ((e = cudaEventRecord(c->ev_bp_join[i], c->bp[i])) != cudaSuccess) return e;
    if ((e = cudaStreamWaitEvent(st, c->ev_bp_join[i], 0)) != cudaSuccess) return e;
  }
  k_uspec<<<dim3((c->s_bins + kN2 - 1) / kN2, count), 256, 0, st>>>(meta, wbuf, ubuf, p);
  c->launches++;
  return cudaGetLastError();
}

}  // namespace gwmf
