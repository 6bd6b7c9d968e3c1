// pass1.cu -- correlate (step a2) and the first pass of the band inverse FFTs (first half of a3).
//
// Index algebra.  n = n1 * 1024.  Input bin k = 1024 k1 + k2, k2 = 32 m + c; output sample j = j1 + n1 j2,
// j2 = jm + 32 jc.
//   z_l[j1 + n1 (jm + 32 jc)] = sum_c e^{2 pi i jc c/32} e^{2 pi i jm c/1024} A_l[j1][c][jm]          (pass 2)
//   A_l[j1][c][jm]  = sum_m e^{2 pi i jm m/32} Y_l[j1][32 m + c]                            (row stage, this file)
//   Y_l[j1][k2]     = e^{2 pi i j1 k2/n} sum_{k1 in band l} Q[1024 k1 + k2] e^{2 pi i j1 k1/n1}  (column transform)
// What this pass leaves in HBM is A_l (p * n complex per template): each row j1 is 8 KB, [c][jm].
// The n1-point column transform is itself split n1 = NA * NB with k1 = NB a + b, j1 = ja + NA jb:
//   stage 1:  V[ja][b] = sum_a Q[NB a + b] w_NA^{ja a}, times e^{2 pi i ja (1024 b + k2)/n}
//   stage 2:  Y[ja + NA jb] = e^{2 pi i NA jb k2/n} sum_b w_NB^{jb b} V[ja][b]
// A band is a contiguous run of bins, i.e. of rows k1, so the transform is pruned to the rows the band touches.
// Kernels:  k_correlate (Q once per template and bin), k_pass1_narrow (bands of <= 32 rows: column transform +
// row stage in one CTA, writes A directly), k_pass1 (generic: wide bands and the dense transform, plain layout
// Y) followed by k_rowstage (Y -> A in place).
#include <limits.h>

#include "fft_reg.cuh"
#include "gwmf_internal.cuh"

namespace gwmf {

struct P1Args {
  const TemplateMeta* meta;   // already offset to the first template of the batch
  const float2* wq;           // weighted spectrum, n/2
  const double* u_tab;        // f^(-1/3), n/2
  const float2* tw_n1;        // e^{2 pi i m/n1}
  const float2* tw_p2;        // [32][32] e^{2 pi i a b/1024}
  const float2* q;            // [batch][n/2] correlated spectrum Q_I[k] (k_correlate)
  const float2* dense_in;     // DENSE only: n complex inputs
  float2* y;                  // [batch][p][n1][1024]: row j1 of band l, A layout [c][jm] (generic kernel: plain Y[k2])
  int p;
  int log_n;
  int n1;
  int batch;                  // templates in this launch
  // decimated path (effective bands, gwmf_internal.cuh): the band buffer is indexed by slot = eff_prefix - slot_base + e
  int slot_base;              // eff_prefix of the first template of the batch
  int first_template;         // bank index of the first template of the batch
  int ja_per_cta;             // k_pass1_eff: consecutive ja values a CTA walks over
  const float2* ubuf;         // [batch][kUCap] one-sided power spectra U+ (bandpower.cu)
  const float2* vbuf;         // [slots][n] pre-passed bands (k_prepass)
};

__device__ __forceinline__ float2 cis_frac(unsigned num, int log_n) {
  // e^{2 pi i num / 2^log_n}, num < 2^log_n <= 2^22: the argument 2 num / n is exact in fp32
  float s, c;
  sincospif(2.0f * (float)num / (float)(1u << log_n), &s, &c);
  return make_float2(c, s);
}

template <int NA, int NB, bool DENSE>
__global__ void __launch_bounds__(256, 2) k_pass1(P1Args a) {
  constexpr int FR = NA >= 32 ? 32 : NA;        // stage-1 transform length = ja outputs per CTA
  constexpr int G = NA / FR;                    // residues r of ja = G m + r
  constexpr int C = kColsPerCta;
  constexpr int SROW = NB * C + C;              // padded stride of S[m][..] in float2
  constexpr int TILES = kN2 / C;

  extern __shared__ float2 smem[];
  float2* S = smem;                             // [FR][SROW]
  float2* A = S + FR * SROW;                    // [FR][C]   e^{2 pi i ja k2/n}
  float2* Bt = A + FR * C;                      // [NB][C]   e^{2 pi i NA jb k2/n}
  __shared__ int s_list[DENSE ? 1 : kMaxBatch * kMaxBands];
  __shared__ int s_cnt[kMaxBatch + 1];

  // work list: the wide bands of the batch (DENSE: the one dense transform); every CTA builds the same list
  int n_list = 1;
  if constexpr (!DENSE)
    n_list = build_wide_list(a.meta, a.batch, a.p, s_list, s_cnt);

  const int tid = threadIdx.x;
  const int x = tid >> 3, c = tid & 7;
  const unsigned nmask = (1u << a.log_n) - 1u;
  const int n1 = a.n1;
  const int n_items = n_list * TILES * G;

#pragma unroll 1
  for (int item = blockIdx.x; item < n_items; item += gridDim.x) {
    const int tile = item % TILES, r = (item / TILES) % G;
    const int band_index = DENSE ? 0 : s_list[item / (TILES * G)];      // tb * p + l
    const int k2 = tile * C + c;

    int e_lo, e_hi, tb_q = 0;
    if constexpr (DENSE) {
      e_lo = 0;
      e_hi = 1 << a.log_n;
    } else {
      const int tb = band_index / a.p, l = band_index - tb * a.p;
      const TemplateMeta* m = a.meta + tb;
      e_lo = m->edges[l];
      e_hi = m->edges[l + 1];
      tb_q = tb;
    }
    // rows and a-range touched by the band (uniform over the CTA)
    const int row_lo = e_lo >> kLogN2, row_hi = (e_hi - 1) >> kLogN2;
    const int a_lo = row_lo / NB, a_hi = (e_hi > e_lo) ? row_hi / NB : -1;

    if (x < FR) A[x * C + c] = cis_frac(((unsigned)((G * x + r) * k2)) & nmask, a.log_n);
    if (x < NB) Bt[x * C + c] = cis_frac(((unsigned)(NA * x) * (unsigned)k2) & nmask, a.log_n);
    __syncthreads();

    // ---------------------------------------------------------------- stage 1: thread (b = x, c)
    // V[ja][b] = sum_a Q[NB a + b] w_NA^{ja a} with ja = G m + r, a = a' + FR g:  w_NA^{ja a} = w_FR^{m a'} w_NA^{r a},
    // so the G inputs that share a' are combined first and ONE FR-point transform over a' follows.
    if (x < NB) {
      const int b = x;
      float2 xin[FR];
#pragma unroll
      for (int ap = 0; ap < FR; ++ap) {
        float2 sum = make_float2(0.f, 0.f);
#pragma unroll
        for (int g = 0; g < G; ++g) {
          const int aa = ap + FR * g;
          const int k = ((NB * aa + b) << kLogN2) + k2;
          if (aa >= a_lo && aa <= a_hi && k >= e_lo && k < e_hi) {
            float2 q;
            if constexpr (DENSE) {
              q = a.dense_in[k];
            } else {
              q = a.q[(size_t)tb_q * (size_t)(1u << (a.log_n - 1)) + k];      // Q_I[k] from k_correlate
            }
            if constexpr (G > 1) {
              if (r > 0) q = cmul(q, a.tw_n1[(r * aa * NB) % n1]);         // w_NA^{r a}
            }
            sum = cadd(sum, q);
          }
        }
        xin[ap] = sum;
      }
      fft_dif<FR>(xin);
#pragma unroll
      for (int m = 0; m < FR; ++m) {
        const int ja = G * m + r;
        const float2 tw = cmul(a.tw_n1[(ja * b) % n1], A[m * C + c]);   // e^{2 pi i ja (1024 b + k2)/n}
        S[m * SROW + b * C + c] = cmul(xin[brev<FR>(m)], tw);
      }
    }
    __syncthreads();

    // ---------------------------------------------------------------- stage 2: thread (m = x, c)
    if (x < FR) {
      const int m = x;
      float2 v[NB];
#pragma unroll
      for (int b = 0; b < NB; ++b) v[b] = S[m * SROW + b * C + c];
      fft_dif<NB>(v);
      {
        float2* out = a.y + ((size_t)band_index * n1 + (size_t)(G * m + r)) * kN2 + k2;
#pragma unroll
        for (int jb = 0; jb < NB; ++jb)
          out[(size_t)jb * NA * kN2] = cmul(v[brev<NB>(jb)], Bt[jb * C + c]);
      }
    }
    __syncthreads();                            // S, A, Bt are rewritten by the next item
  }
}


// ---------------------------------------------------------------------------------------------------
// Row stage for the rows written by k_pass1 in the plain layout Y[j1][k2]: first 32-point stage of the
// 1024-point row transform, in place,
//     A[j1][c][jm] = sum_m e^{2 pi i jm m/32} Y[j1][32 m + c],
// which is the layout pass 2 reads (k_pass1_narrow writes it directly).  One warp per row; only the
// bands in the wide list (or every band if use_mask == 0: small n, dense transform) are touched.
// ---------------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(256) k_rowstage(float2* __restrict__ y, const float2* __restrict__ tw_p2,
                                                  const TemplateMeta* __restrict__ meta, int batch, int p, int log_n1,
                                                  int n_bands_all, int use_mask) {
  // use_mask: 0 = every band, 1 = the wide bands (wide_mask)
  __shared__ int s_list[kMaxBatch * kMaxBands];
  __shared__ int s_cnt[kMaxBatch + 1];
  const int n_list = use_mask ? build_wide_list(meta, batch, p, s_list, s_cnt) : n_bands_all;
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  const long long total_rows = (long long)n_list << log_n1;
  for (long long row = (long long)blockIdx.x * 8 + warp; row < total_rows; row += (long long)gridDim.x * 8) {
    const int w = (int)(row >> log_n1), j1 = (int)(row & ((1 << log_n1) - 1));
    const int band = use_mask ? s_list[w] : w;
    float2* Y = y + (((size_t)band << log_n1) + (size_t)j1) * kN2;
    float2 x[32];
#pragma unroll
    for (int m = 0; m < 32; ++m) x[brev<32>(m)] = Y[32 * m + lane];       // lane = c
    fft_dit<32>(x);                                                        // over m -> jm
    __syncwarp();                                                          // the whole row is in registers
    float4* out = reinterpret_cast<float4*>(Y + 32 * lane);
#pragma unroll
    for (int jm = 0; jm < 32; jm += 2) out[jm >> 1] = make_float4(x[jm].x, x[jm].y, x[jm + 1].x, x[jm + 1].y);
  }
}


// ---------------------------------------------------------------------------------------------------
// Correlate (step a2): Q_I[k] = w[k] e^{i Psi0_I(f_k)} for k_low <= k < k_high, once per (template, bin).
// The phase is evaluated in fp64 (Horner in u = f^(-1/3), coefficients in turns), reduced to one turn in
// fp64, and only then rounded to fp32 for sincospif.  Q (4 MiB per template at n = 2^20) is written once and
// read by every ja-slice of pass 1 out of L2.
// ---------------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(256) k_correlate(const TemplateMeta* __restrict__ meta, const float2* __restrict__ wq,
                                                   const double* __restrict__ u_tab, float2* __restrict__ q, int half_n,
                                                   int k_first) {
  const TemplateMeta* m = meta + blockIdx.y;
  const int k = k_first + blockIdx.x * 256 + threadIdx.x;
  if (k < m->edges[0] || k >= m->k_high) return;
  // correlate: template phasor times weighted data bin (Eq. 1 integrand)
  const double u = u_tab[k];
  double t = fma(fma(fma(fma(m->c0, u * u, m->c2), u, m->c3), u, m->c4), u, -0.125);   // Psi0 / 2 pi, turns
  t -= rint(t);
  float sn, cs;
  sincospif(2.0f * (float)t, &sn, &cs);
  q[(size_t)blockIdx.y * half_n + k] = cmul(wq[k], make_float2(cs, sn));
}

// The same values with every row of 1024 bins stored C-MAJOR (bin 32 m + c at position 32 c + m, cm_pos): the layout
// the decimated path's first pass reads with lane = m.  One CTA per (row, template); the row is transposed through
// shared memory so that both the reads of wq / u_tab and the writes of Q are coalesced.
__global__ void __launch_bounds__(256) k_correlate_cm(const TemplateMeta* __restrict__ meta, const float2* __restrict__ wq,
                                                      const double* __restrict__ u_tab, float2* __restrict__ q, int half_n,
                                                      int row_first) {
  __shared__ float2 sq[kN2 + 32];
  const TemplateMeta* m = meta + blockIdx.y;
  const int row = row_first + blockIdx.x;
  const int k_lo = m->edges[0], k_hi = m->k_high;
  if ((row + 1) * kN2 <= k_lo || row * kN2 >= k_hi) return;            // CTA-uniform
  const double c0 = m->c0, c2 = m->c2, c3 = m->c3, c4 = m->c4;
#pragma unroll
  for (int i = 0; i < 4; ++i) {
    const int k2 = threadIdx.x + 256 * i, k = row * kN2 + k2;
    float2 v = make_float2(0.f, 0.f);
    if (k >= k_lo && k < k_hi) {
      // correlate: template phasor times weighted data bin (Eq. 1 integrand)
      const double u = u_tab[k];
      double t = fma(fma(fma(fma(c0, u * u, c2), u, c3), u, c4), u, -0.125);   // Psi0 / 2 pi, turns
      t -= rint(t);
      float sn, cs;
      sincospif(2.0f * (float)t, &sn, &cs);
      v = cmul(wq[k], make_float2(cs, sn));
    }
    const int pos = cm_pos(k2);
    sq[pos + (pos >> 5)] = v;
  }
  __syncthreads();
  float2* out = q + (size_t)blockIdx.y * half_n + (size_t)row * kN2;
#pragma unroll
  for (int i = 0; i < 4; ++i) {
    const int pos = threadIdx.x + 256 * i, k = row * kN2 + cm_pos(pos);
    if (k >= k_lo && k < k_hi) out[pos] = sq[pos + (pos >> 5)];
  }
}

// ---------------------------------------------------------------------------------------------------
// Narrow bands (at most 32 input rows: 99 % of the bands of the headline bank).  n1 = NA * 32, output row
// j1 = ja + NA jb, input row k1 = 32 a + b.  With so few rows every residue b has at most one non-zero
// input, so the transform over a degenerates to the single product Q[k] e^{2 pi i ja k/n}, and the band's
// rows, rotated so that the first one sits at b' = 0, feed a 32-point transform over b whose zero tail is
// pruned at compile time (RMAX = 4, 8, 16, 32).
//
// A CTA owns one ja and the 256 columns k2 = 32 m + c, m = 0..31, c = 8 cg .. 8 cg + 7, and runs both the
// column transform and the first stage of the row transform (over m), so that what reaches HBM is already
//     A[j1][c][jm] = sum_m e^{2 pi i jm m/32} Y[j1][32 m + c],
// the layout pass 2 consumes with one twiddle and one 32-point transform per thread:
//   phase 1, thread (m, ci):  v[jb] = FFT32_b( Q[k] e^{2 pi i ja k/n} ),  tile[jb][m][ci] = v[jb] e^{2 pi i jb m/1024}
//   phase 2, thread (jb, ci): x[m] = tile[jb][m][ci] S,  S = e^{2 pi i jb (c + 1024 b0)/32768}  (the rest of the
//                             column twiddle e^{2 pi i NA jb k2/n} and the rotation w_32^{jb b0});
//                             X[jm] = FFT32_m(x);  staged as [jb][ci][jm]
//   store: per jb one contiguous 2 KB piece of row j1, by TMA bulk copy shared -> global.
// ---------------------------------------------------------------------------------------------------
constexpr int kTileStride = 257;      // float2 per jb row of the exchange tile (conflict-free both ways)
constexpr int kStageStride = 258;     // float2 per jb row of the store staging (16-byte aligned rows)
constexpr int kT1Stride = 34;         // float2 per row of the shared twiddle table (16-byte aligned, conflict-free LDS.128)

template <int RMAX>
__device__ __forceinline__ void narrow_phase1(const P1Args& a, const float2* __restrict__ qrow, const float2* __restrict__ T1,
                                              float2* __restrict__ tile, float2 Aja, int R, int row_lo, int e_lo, int e_hi,
                                              int ja, int k2, int m, int ci) {
  float2 v[32];
  const int n1m = a.n1 - 1;
#pragma unroll
  for (int i = 0; i < RMAX; ++i) {
    float2 val = make_float2(0.f, 0.f);
    const int k = ((row_lo + i) << kLogN2) + k2;
    if (i < R && k >= e_lo && k < e_hi) {
      const float2 t = cmul(a.tw_n1[(ja * (row_lo + i)) & n1m], Aja);      // e^{2 pi i ja k/n}, k = 1024 k1 + k2
      val = cmul(qrow[k], t);
    }
    v[brev<32>(i)] = val;
  }
  fft_dit<32, RMAX>(v);                     // inputs i >= RMAX are zero: leading stages pruned
  // T1 is symmetric: row m holds e^{2 pi i jb m/1024} for consecutive jb, read two at a time
  const float4* __restrict__ t1 = reinterpret_cast<const float4*>(T1 + m * kT1Stride);
#pragma unroll
  for (int jb = 0; jb < 32; jb += 2) {
    const float4 w = t1[jb >> 1];
    tile[jb * kTileStride + m * 8 + ci] = cmul(v[jb], make_float2(w.x, w.y));
    tile[(jb + 1) * kTileStride + m * 8 + ci] = cmul(v[jb + 1], make_float2(w.z, w.w));
  }
}

__global__ void __launch_bounds__(256, 3) k_pass1_narrow(P1Args a) {
  extern __shared__ __align__(128) float2 smem[];
  float2* tile = smem;                          // [32][kStageStride] (phase 1 uses stride kTileStride)
  float2* T1 = smem + 32 * kStageStride;        // [32 m][kT1Stride]  e^{2 pi i jb m/1024}

  const int tid = threadIdx.x;
  const int na = a.n1 >> 5;
  const int cg = blockIdx.x & 3, ja = blockIdx.x >> 2;
  const int l = blockIdx.y, tb = blockIdx.z;
  const int band_index = tb * a.p + l;
  const unsigned nmask = (1u << a.log_n) - 1u;

  const TemplateMeta* mt = a.meta + tb;
  const int e_lo = mt->edges[l], e_hi = mt->edges[l + 1];
  float2* out0 = a.y + ((size_t)band_index * a.n1 + (size_t)ja) * kN2 + cg * 256;   // row jb adds jb * na * 1024
  const size_t row_stride = (size_t)na * kN2;
  if (e_hi <= e_lo) {             // empty band: z_l = 0
#pragma unroll 4
    for (int jb = 0; jb < 32; ++jb) out0[(size_t)jb * row_stride + tid] = make_float2(0.f, 0.f);
    return;
  }
  const int row_lo = e_lo >> kLogN2, row_hi = (e_hi - 1) >> kLogN2;
  const int R = row_hi - row_lo + 1;
  if (R > 32) return;             // wide band: k_pass1 + k_rowstage

#pragma unroll
  for (int i = 0; i < 4; ++i) T1[(tid >> 5) * kT1Stride + 8 * i * kT1Stride + (tid & 31)] = __ldg(&a.tw_p2[tid + 256 * i]);
  __syncthreads();
  // ---- phase 1: thread (m, ci), column k2
  {
    const int ci = tid & 7, m = tid >> 3;
    const int k2 = 32 * m + 8 * cg + ci;
    const float2 Aja = cis_frac(((unsigned)ja * (unsigned)k2) & nmask, a.log_n);
    const float2* qrow = a.q + (size_t)tb * (size_t)(1u << (a.log_n - 1));
    if (R <= 4) narrow_phase1<4>(a, qrow, T1, tile, Aja, R, row_lo, e_lo, e_hi, ja, k2, m, ci);
    else if (R <= 8) narrow_phase1<8>(a, qrow, T1, tile, Aja, R, row_lo, e_lo, e_hi, ja, k2, m, ci);
    else if (R <= 16) narrow_phase1<16>(a, qrow, T1, tile, Aja, R, row_lo, e_lo, e_hi, ja, k2, m, ci);
    else narrow_phase1<32>(a, qrow, T1, tile, Aja, R, row_lo, e_lo, e_hi, ja, k2, m, ci);
  }
  __syncthreads();
  // ---- phase 2: thread (jb = lane, ci = warp)
  {
    const int jb = tid & 31, ci = tid >> 5;
    const int c = 8 * cg + ci;
    float sn, cs;
    const unsigned num = ((unsigned)jb * (unsigned)(c + 1024 * (row_lo & 31))) & 32767u;
    sincospif((float)num * (1.0f / 16384.0f), &sn, &cs);
    const tw4 S = make_tw4(make_float2(cs, sn));
    float2 x[32];
#pragma unroll
    for (int m = 0; m < 32; ++m) x[brev<32>(m)] = cmul_tw(tile[jb * kTileStride + m * 8 + ci], S);
    fft_dit<32>(x);                                   // over m -> jm
    __syncthreads();                                  // the tile has been read by everyone: reuse it as staging
    float4* st = reinterpret_cast<float4*>(tile + jb * kStageStride + ci * 32);
#pragma unroll
    for (int jm = 0; jm < 32; jm += 2) st[jm >> 1] = make_float4(x[jm].x, x[jm].y, x[jm + 1].x, x[jm + 1].y);
  }
  asm volatile("fence.proxy.async.shared::cta;" ::: "memory");     // generic writes -> visible to the bulk copy engine
  __syncthreads();
  if (tid < 32) {
    const unsigned src = (unsigned)__cvta_generic_to_shared(tile + tid * kStageStride);
    float2* dst = out0 + (size_t)tid * row_stride;
    asm volatile("cp.async.bulk.global.shared::cta.bulk_group [%0], [%1], 2048;" ::"l"(dst), "r"(src) : "memory");
    asm volatile("cp.async.bulk.commit_group;" ::: "memory");
    asm volatile("cp.async.bulk.wait_group.read 0;" ::: "memory");   // shared memory must outlive the copy's reads
  }
}

// ---------------------------------------------------------------------------------------------------
// Decimated path: first pass of the n-point transform of an EFFECTIVE band (gwmf_internal.cuh: Z = union of the
// narrow bands read from Q, U = one-sided power spectrum read from ubuf, D = one wide band read from Q), any number
// of input rows.  WARP-AUTONOMOUS: a CTA owns one ja and 8 values of c (one per warp); a warp owns the 32 columns
// k2 = 32 m + c, m = lane, and runs both the column transform and the first stage of the row transform on them
// with no CTA barrier at all:
//   phase 1, lane = m:  for every residue b' = (k1 - row_lo) mod 32, with k1 = row_lo + b' + 32 t,
//         v[b'] = TW[b'] sum_t X[k1][k2] g^t,   g = e^{2 pi i ja/NA},  TW[i] = e^{2 pi i ja (row_lo + i)/n1}
//       (Horner's rule over the rounds t, highest first; bands of <= 16 rows use pruned variants), then the 32-point
//       transform over b' -> jb, and the lane writes ITS column of the warp's 32 x 32 tile.
//   phase 2, lane = jb: reads ITS row of the tile (all m), multiplies by the twiddle
//         e^{2 pi i [c j1 + (n/32) jb b0 + (jb n1 + 32 ja) m]/n} = S w^m,   j1 = ja + NA jb, b0 = row_lo mod 32
//       (column twiddle e^{2 pi i j1 k2/n}, rotation w_32^{jb b0}, and the twiddle between the two 32-point stages of
//       the row transform; geometric in m: w^m = w8^(m >> 3) w^(m & 7), two exact angles per lane, no table),
//       32-point transform over m -> jm, and stages the 256 B piece A[j1][c][0..31] in the SAME row of the tile, from
//       where one bulk copy (cp.async.bulk shared -> global, issued by the lane itself) takes it to the band buffer.
// A lane only ever re-writes tile cells it was the last to read, so one __syncwarp() between the phases is all the
// synchronisation there is.  The input spectra are stored C-MAJOR inside each row of 1024 bins (bin 32 m + c at
// position 32 c + m, cm_pos) so that the 32 lanes of a warp read 256 contiguous bytes.
// Bins of class-D bands that lie inside the hull of Z ("holes": only with unusual spectra) are masked out.
// ---------------------------------------------------------------------------------------------------
struct EffSrc {
  const float2* src;      // spectrum, rows of 1024 bins in c-major order: bin k at src[(k & ~1023) + cm_pos(k & 1023)]
  int e_lo, e_hi;
  int n_holes;            // Z only
  const int* holes;       // shared memory: [2h] = first bin of hole h, [2h+1] = one past its last bin
  const float2* v;        // pre-passed band (k_prepass): V of this slot, else nullptr
};

// A warp's tile: 32 rows (jb) of 256 B, no padding; the 16-byte chunk ch of row r sits at chunk ch ^ (r & 15), which
// makes the column writes of phase 1, the row reads / writes of phase 2 (16 bytes per lane) and the bulk copy's linear
// read all conflict-free.  The tile reaches the band buffer as it is (pass 2 undoes the swizzle when it reads).
constexpr int kWTile = 32 * 32;                   // float2 per warp (8 KB)
// Measured on B200 (headline config): 4 warps x 4 CTAs per SM at 128 registers (ptxas: 28 B spill stores, 36 B spill
// loads per thread) beats 8 x 3 at 80 registers
// (spills in the round loop) by 20 %; 2..8 ja per CTA are within 2 % of each other, 1 and 32 are worse.
constexpr int kP1Warps = 4;                       // warps (values of c) per CTA of k_pass1_eff
constexpr int kP1CtasPerSm = 4;
constexpr int kP1JaPerCta = 4;                    // consecutive ja a CTA walks over
constexpr int kP1Groups = 32 / kP1Warps;          // CTAs (column groups cg) per ja
constexpr size_t kP1WSmem = (size_t)(kP1Warps * kWTile + kP1Warps * 64) * sizeof(float2);     // tiles + per-warp TW tables {w, i w}

// 16-byte shared-memory access at (addr ^ x): the XOR is part of the asm so that the 16 addresses of a row are formed
// where they are used instead of being kept in registers
__device__ __forceinline__ float4 lds128_x(unsigned addr, unsigned x) {
  float4 v;
  asm volatile("{\n\t.reg .u32 a;\n\txor.b32 a, %4, %5;\n\tld.shared.v4.f32 {%0, %1, %2, %3}, [a];\n\t}"
               : "=f"(v.x), "=f"(v.y), "=f"(v.z), "=f"(v.w)
               : "r"(addr), "r"(x));
  return v;
}
__device__ __forceinline__ void sts128_x(unsigned addr, unsigned x, float4 v) {
  asm volatile("{\n\t.reg .u32 a;\n\txor.b32 a, %0, %1;\n\tst.shared.v4.f32 [a], {%2, %3, %4, %5};\n\t}" ::"r"(addr), "r"(x),
               "f"(v.x), "f"(v.y), "f"(v.z), "f"(v.w)
               : "memory");
}
// 8-byte store to cell (row i, element m = lane) of a warp's swizzled tile: byte address ((col ^ x) + off) with
// col = tile | lane * 8, x = (i & 15) << 4, off = i * 256 (the XOR and the offset are part of the asm: nothing is hoisted)
__device__ __forceinline__ void sts64_xo(unsigned col, unsigned x, unsigned off, float2 v) {
  asm volatile("{\n\t.reg .u32 a;\n\txor.b32 a, %0, %1;\n\tadd.u32 a, a, %2;\n\tst.shared.v2.f32 [a], {%3, %4};\n\t}" ::"r"(col), "r"(x),
               "r"(off), "f"(v.x), "f"(v.y)
               : "memory");
}

template <bool HOLES>
__device__ __forceinline__ bool eff_ok(const EffSrc& es, int k1, int k2, int fr, int lr) {
  bool ok = k1 >= fr && k1 <= lr;
  if constexpr (HOLES) {
    const int k = k1 * kN2 + k2;
    for (int h = 0; h < es.n_holes; ++h) ok = ok && !(k >= es.holes[2 * h] && k < es.holes[2 * h + 1]);
  }
  return ok;
}

// predicated 8-byte load (no branch): 0 where !ok
__device__ __forceinline__ float2 ldg_pred(const float2* p, bool ok) {
  float2 v = make_float2(0.f, 0.f);
  asm("{\n\t.reg .pred p;\n\tsetp.ne.s32 p, %3, 0;\n\t@p ld.global.nc.v2.f32 {%0, %1}, [%2];\n\t}"
      : "+f"(v.x), "+f"(v.y)
      : "l"(p), "r"((int)ok));
  return v;
}


// Phase 1 of a warp (lane = m, column k2 = 32 lane + c): leaves v[jb], jb = 0..31 in natural order.  Registers and global
// loads only.  TW: the warp's table (shared).
template <int RMAX, bool HOLES>
__device__ __forceinline__ void eff_phase1(const P1Args& a, const EffSrc& es, const float4* __restrict__ TW,
                                           int ja, int c, int lane, float2 (&v)[32]) {
  const int row_lo = es.e_lo >> kLogN2, row_hi = (es.e_hi - 1) >> kLogN2;
  const int R = row_hi - row_lo + 1;
  const int T = RMAX < 32 ? 1 : es.v ? a.n1 >> 10 : (R + 31) >> 5;    // pre-passed band: Q = NA / 32 rounds, every row of V valid
  const int k2 = 32 * lane + c;
  const int fr = es.v ? INT_MIN : row_lo + (k2 < (es.e_lo & (kN2 - 1)) ? 1 : 0);       // first / last row whose bin in THIS column is in the band
  const int lr = es.v ? INT_MAX : row_hi - (k2 > ((es.e_hi - 1) & (kN2 - 1)) ? 1 : 0);
  const float2* __restrict__ base = es.src + c * 32 + lane;            // + k1 * 1024 (k1 < 0 in the lower half of a pair spectrum)

  // rows of round t: the band's rows row_lo + 32 t + i, or (pre-passed band, es.v != nullptr) the 32 rows b' = i of V[t][ja mod 32]
  auto round_ptr = [&](int t) -> const float2* {
    return es.v ? es.v + ((size_t)(t * 32 + (ja & 31)) * 32) * kN2 + c * 32 + lane : base + (ptrdiff_t)(row_lo + 32 * t) * kN2;
  };
  // top round (t = T - 1) straight into the registers of the transform
  {
    const int r0 = row_lo + 32 * (T - 1);
    const float2* __restrict__ p0 = round_ptr(T - 1);
#pragma unroll
    for (int i = 0; i < RMAX; ++i) {
      const bool ok = eff_ok<HOLES>(es, r0 + i, k2, fr, lr);
      v[brev<32>(i)] = ldg_pred(p0 + i * kN2, ok);
    }
  }
  if constexpr (RMAX == 32) {
    if (T > 1) {
      // The rounds below the top one, highest first: v = v g + X_t (Horner), the rows of a round loaded in groups of 8
      // straight into registers, two groups in flight while the one before them is consumed (no shared-memory staging:
      // the L1 data pipe is this kernel's busiest unit).
      auto load_group = [&](int t, int gq, float2 (&dst)[8]) {
        const int r0 = row_lo + 32 * t + 8 * gq;
        const float2* __restrict__ p0 = round_ptr(t) + (size_t)(8 * gq) * kN2;
#pragma unroll
        for (int j = 0; j < 8; ++j) dst[j] = ldg_pred(p0 + j * kN2, eff_ok<HOLES>(es, r0 + j, k2, fr, lr));
      };
      const float2 g1 = a.tw_n1[(ja * 32) & (a.n1 - 1)];                          // e^{2 pi i ja/NA}
      const pk2 g = pk(g1), ig = pk(-g1.y, g1.x);
      float2 bufA[8], bufB[8];                      // two groups in flight: A holds the even groups of a round, B the odd ones
      load_group(T - 2, 0, bufA);
      load_group(T - 2, 1, bufB);
      auto consume = [&](int gq, const float2 (&cur)[8]) {
#pragma unroll
        for (int j = 0; j < 8; ++j) {
          const float2 w = v[brev<32>(8 * gq + j)];
          v[brev<32>(8 * gq + j)] = unpk(fma2(pk(w.y, w.y), ig, fma2(pk(w.x, w.x), g, pk(cur[j]))));   // v g + X = w.x g + w.y (i g) + X
        }
      };
#pragma unroll 1
      for (int t = T - 2; t >= 0; --t) {
        consume(0, bufA);
        load_group(t, 2, bufA);
        consume(1, bufB);
        load_group(t, 3, bufB);
        consume(2, bufA);
        if (t > 0) load_group(t - 1, 0, bufA);
        consume(3, bufB);
        if (t > 0) load_group(t - 1, 1, bufB);
      }
    }
  }
#pragma unroll
  for (int i = 0; i < RMAX; ++i) {                 // v w = v.x w + v.y (i w): no negation of the data
    const float4 w = TW[i];
    const float2 x = v[brev<32>(i)];
    v[brev<32>(i)] = unpk(fma2(pk(x.y, x.y), pk(w.z, w.w), mul2(pk(x.x, x.x), pk(w.x, w.y))));
  }
  fft_dit<32, RMAX>(v);                     // inputs i >= RMAX are zero: leading stages pruned
}

template <bool HOLES>
__device__ __forceinline__ void eff_warp(const P1Args& a, const EffSrc& es, const float4* TW, int ja, int c, int lane,
                                         float2 (&v)[32]) {
  const int R = ((es.e_hi - 1) >> kLogN2) - (es.e_lo >> kLogN2) + 1;
  // two pruned variants: more of them cost more in instruction-cache misses than their shorter transforms save
  if (R <= 16) eff_phase1<16, HOLES>(a, es, TW, ja, c, lane, v);
  else eff_phase1<32, HOLES>(a, es, TW, ja, c, lane, v);
}

__global__ void __launch_bounds__(kP1Warps * 32, kP1CtasPerSm) k_pass1_eff(P1Args a, const SlotDesc* __restrict__ slot_tab) {
  extern __shared__ __align__(1024) float2 smem[];
  __shared__ int s_holes[2 * kMaxBands];

  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  float2* tile = smem + warp * kWTile;          // this warp's swizzled [32][32] tile (wz)
  float4* TW = reinterpret_cast<float4*>(smem + kP1Warps * kWTile) + warp * 32;   // this warp's {w, i w}, w = e^{2 pi i ja (row_lo + i)/n1}
  const int na = a.n1 >> 5, n1m = a.n1 - 1;
  const int cg = blockIdx.x % kP1Groups, ja0 = (blockIdx.x / kP1Groups) * a.ja_per_cta;
  const int ja1 = ja0 + a.ja_per_cta < na ? ja0 + a.ja_per_cta : na;
  const int c = kP1Warps * cg + warp;
  const int slot = blockIdx.y;                  // batch-relative
  const unsigned nmask = (1u << a.log_n) - 1u;

  const SlotDesc d = slot_tab[a.slot_base + slot];      // one 32-byte load, same address in every thread
  const int tb = d.t - a.first_template;

  EffSrc es;
  es.v = d.generic ? a.vbuf + ((size_t)slot << a.log_n) : nullptr;      // very many rows: reduced to Q rounds by k_prepass
  es.e_lo = d.e_lo;
  es.e_hi = d.e_hi;
  es.holes = s_holes;
  es.n_holes = d.n_holes;
  es.src = d.kind == kEffU    ? a.ubuf + (size_t)tb * kUCap
           : d.kind == kEffUP ? a.ubuf + (size_t)(tb + 1) * kUCap              // bin 0 of the pair spectrum; bins run negative
                              : a.q + (size_t)tb * (size_t)(1u << (a.log_n - 1));
  const int row_lo = es.e_lo >> kLogN2;
  if (d.n_holes > 0) {                          // rare: class-D bands inside the hull of Z (CTA-uniform branch)
    if (tid == 0) {
      const TemplateMeta* mt = a.meta + tb;
      int nh = 0;
      unsigned dm = mt->d_mask;
      while (dm) {
        const int l = __ffs(dm) - 1;
        dm &= dm - 1;
        if (mt->edges[l] >= es.e_lo && mt->edges[l + 1] <= es.e_hi) { s_holes[2 * nh] = mt->edges[l]; s_holes[2 * nh + 1] = mt->edges[l + 1]; ++nh; }
      }
    }
    __syncthreads();
  }
  // The warp walks over its ja values.  The bulk store of a tile is only waited for when the tile is written again,
  // after the next ja's first 32-point transform; TW of the next ja is fetched one iteration ahead.
  float2 tw_next = __ldg(&a.tw_n1[(ja0 * (row_lo + lane)) & n1m]);
#pragma unroll 1
  for (int ja = ja0; ja < ja1; ++ja) {
  TW[lane] = make_float4(tw_next.x, tw_next.y, -tw_next.y, tw_next.x);
  __syncwarp();
  if (ja + 1 < ja1) tw_next = __ldg(&a.tw_n1[((ja + 1) * (row_lo + lane)) & n1m]);
  float2 v[32];
  if (d.n_holes > 0) eff_warp<true>(a, es, TW, ja, c, lane, v);
  else eff_warp<false>(a, es, TW, ja, c, lane, v);
  // the previous ja's bulk store must have read the tile before it is written again
  if (lane == 0) asm volatile("cp.async.bulk.wait_group.read 0;" ::: "memory");
  __syncwarp();
  // the lane's column of the tile: tile[jb][m = lane]
  const unsigned col = (unsigned)__cvta_generic_to_shared(tile) | ((unsigned)lane << 3);
#pragma unroll
  for (int jb = 0; jb < 32; ++jb) sts64_xo(col, (jb & 15) << 4, jb * 256, v[jb]);
  __syncwarp();

  // ---- phase 2: lane = jb, row j1 = ja + NA jb
  const int jb = lane;
  const unsigned j1 = (unsigned)ja + (unsigned)na * (unsigned)jb;
  // S = e^{2 pi i [c j1 + (n/32) jb b0]/n},  w = e^{2 pi i (jb n1 + 32 ja)/n}: exact angles in integers mod n
  const unsigned num_s = ((unsigned)c * j1 + (((unsigned)jb * (unsigned)(row_lo & 31)) << (a.log_n - 5))) & nmask;
  const unsigned num_w = ((unsigned)jb * (unsigned)a.n1 + 32u * (unsigned)ja) & nmask;
  const float2 S = cis_frac(num_s, a.log_n);
  const float2 w1 = cis_frac(num_w, a.log_n);
  const float2 w8 = cis_frac((8u * num_w) & nmask, a.log_n);
  // W[lo] = w^lo, lo < 8 (chain from w); B[hi] = S w8^hi, hi < 4
  tw4 B[4];
  {
    float2 b = S;
    B[0] = make_tw4(b);
#pragma unroll
    for (int hi = 1; hi < 4; ++hi) { b = cmul(b, w8); B[hi] = make_tw4(b); }
  }
  float2 x[32];
  {
    // chunk ch of the lane's row sits at ch ^ (jb & 15): one XOR on the byte address per access
    const unsigned row = (unsigned)__cvta_generic_to_shared(tile + jb * 32) | ((unsigned)(jb & 15) << 4);
    float2 wl = make_float2(1.f, 0.f);
#pragma unroll
    for (int lo = 0; lo < 8; lo += 2) {
      const tw4 Wa = make_tw4(wl);
      wl = cmul(wl, w1);
      const tw4 Wb = make_tw4(wl);
      if (lo < 6) wl = cmul(wl, w1);
#pragma unroll
      for (int hi = 0; hi < 4; ++hi) {
        const int m = 8 * hi + lo;
        const float4 t = lds128_x(row, (unsigned)(m >> 1) << 4);        // tile[jb][m], tile[jb][m + 1]
        const float2 t0 = make_float2(t.x, t.y), t1 = make_float2(t.z, t.w);
        x[brev<32>(m)] = cmul_tw(lo == 0 ? t0 : cmul_tw(t0, Wa), B[hi]);
        x[brev<32>(m + 1)] = cmul_tw(cmul_tw(t1, Wb), B[hi]);
      }
    }
  }
  fft_dit<32>(x);                                   // over m -> jm
  // stage the 256 B piece A[j1][c][0..31] in the lane's own row of the tile (same swizzle); the whole 8 KB tile then
  // leaves with ONE bulk copy: the band buffer is [slot][ja][c][jb][jm]
  {
    const unsigned row = (unsigned)__cvta_generic_to_shared(tile + jb * 32) | ((unsigned)(jb & 15) << 4);
#pragma unroll
    for (int jm = 0; jm < 32; jm += 2) sts128_x(row, (unsigned)(jm >> 1) << 4, make_float4(x[jm].x, x[jm].y, x[jm + 1].x, x[jm + 1].y));
  }
  asm volatile("fence.proxy.async.shared::cta;" ::: "memory");     // generic writes -> visible to the bulk copy engine
  __syncwarp();
  if (lane == 0) {
    float2* dst = a.y + ((((size_t)slot * na + ja) * 32 + c) << 10);
    const unsigned src = (unsigned)__cvta_generic_to_shared(tile);
    asm volatile("cp.async.bulk.global.shared::cta.bulk_group [%0], [%1], 8192;" ::"l"(dst), "r"(src) : "memory");
    asm volatile("cp.async.bulk.commit_group;" ::: "memory");
  }
  }   // ja
  if (lane == 0) asm volatile("cp.async.bulk.wait_group.read 0;" ::: "memory");   // shared memory must outlive the copy's reads
}

// ---------------------------------------------------------------------------------------------------
// Pre-pass for effective bands of very many input rows (SlotDesc::generic; n1 >= 1024, NA = 32 Q).  The Horner sum
// of k_pass1_eff over the T = ceil(R / 32) rounds t costs T multiply-adds per (ja, b', column) and re-reads the whole
// band for every ja.  With t = t0 + Q t1 and G = e^{2 pi i ja/NA}, G^Q = e^{2 pi i ja/32} depends on ja mod 32 only:
//     sum_t X_t G^t = sum_{t0 < Q} G^{t0} V[t0][ja mod 32],   V[t0][ja1][b'][.] = sum_{t1 < 32} X_{t0 + Q t1}[b'][.] e^{2 pi i ja1 t1/32}
// so ONE 32-point transform per (t0, b', column) serves all ja, and k_pass1_eff is left with Q <= 4 rounds read from
// V (n complex per band: the slot's twin in vbuf, rows c-major like Q).  Thread = (t0, b', position in the row);
// the work items of a batch are listed by k_pp_jobs and walked grid-stride.
// ---------------------------------------------------------------------------------------------------
__global__ void k_pp_jobs(const SlotDesc* __restrict__ slot_tab, int slot_base, int n_slots, int* __restrict__ list,
                          int* __restrict__ n_list) {
  __shared__ int s_n;
  if (threadIdx.x == 0) s_n = 0;
  __syncthreads();
  for (int s = threadIdx.x; s < n_slots; s += blockDim.x)
    if (slot_tab[slot_base + s].generic) list[atomicAdd(&s_n, 1)] = s;       // any order: a band's V is its own
  __syncthreads();
  if (threadIdx.x == 0) *n_list = s_n;
}

__global__ void __launch_bounds__(256) k_prepass(P1Args a, const SlotDesc* __restrict__ slot_tab, float2* __restrict__ vbuf,
                                                  const int* __restrict__ list, const int* __restrict__ n_list) {
  const int na = a.n1 >> 5, Q = na >> 5;
  const int per_band = 4 * 32 * Q;               // CTAs per band: 4 position chunks x 32 b' x Q t0
  const int n_items = *n_list * per_band;
  const size_t n = (size_t)1 << a.log_n;
#pragma unroll 1
  for (int item = blockIdx.x; item < n_items; item += gridDim.x) {
    const int slot = list[item / per_band];
    int rem = item % per_band;
    const int chunk = rem & 3;
    rem >>= 2;
    const int bp = rem & 31, t0 = rem >> 5;
    const SlotDesc d = slot_tab[a.slot_base + slot];
    const int tb = d.t - a.first_template;
    const float2* __restrict__ src = a.q + (size_t)tb * (n >> 1);          // class D (or the whole template): read from Q
    const int row_lo = d.e_lo >> kLogN2, row_hi = (d.e_hi - 1) >> kLogN2;
    const int pos = chunk * 256 + threadIdx.x, k2 = cm_pos(pos);
    const int fr = row_lo + (k2 < (d.e_lo & (kN2 - 1)) ? 1 : 0);           // first / last row whose bin in THIS column is in the band
    const int lr = row_hi - (k2 > ((d.e_hi - 1) & (kN2 - 1)) ? 1 : 0);
    float2 x[32];
#pragma unroll
    for (int t1 = 0; t1 < 32; ++t1) {
      const int k1 = row_lo + bp + 32 * (t0 + Q * t1);
      x[brev<32>(t1)] = ldg_pred(src + (size_t)k1 * kN2 + pos, k1 >= fr && k1 <= lr);
    }
    fft_dit<32>(x);
    float2* __restrict__ out = vbuf + (size_t)slot * n + ((size_t)(t0 * 32) * 32 + bp) * kN2 + pos;
#pragma unroll
    for (int ja1 = 0; ja1 < 32; ++ja1) out[(size_t)ja1 * 32 * kN2] = x[ja1];
  }
}

constexpr size_t kNarrowSmem = (size_t)(32 * kStageStride + 32 * kT1Stride) * sizeof(float2);

static cudaError_t launch_narrow(Ctx* c, const P1Args& args, int batch) {
  dim3 grid(4 * c->na, c->prm.p, batch);
  k_pass1_narrow<<<grid, 256, kNarrowSmem, c->stream>>>(args);
  c->launches++;
  return cudaGetLastError();
}

template <int NA, int NB>
constexpr size_t p1_smem() {
  constexpr int FR = NA >= 32 ? 32 : NA;
  constexpr int SROW = NB * kColsPerCta + kColsPerCta;
  return (size_t)(FR * SROW + FR * kColsPerCta + NB * kColsPerCta) * sizeof(float2);
}

template <int NA, int NB, bool DENSE>
static cudaError_t launch_p1(Ctx* c, const P1Args& args, cudaStream_t st) {
  const size_t smem = p1_smem<NA, NB>();
  // persistent over the work list; a CTA with nothing to do exits after building the (empty) list
  k_pass1<NA, NB, DENSE><<<2 * c->n_sms, 256, smem, st>>>(args);
  c->launches++;
  return cudaGetLastError();
}

template <bool DENSE>
static cudaError_t dispatch_p1(Ctx* c, const P1Args& args, cudaStream_t st) {
  switch (c->na) {
    case 1:
      if (c->nb == 16) return launch_p1<1, 16, DENSE>(c, args, st);
      return launch_p1<1, 32, DENSE>(c, args, st);
    case 2: return launch_p1<2, 32, DENSE>(c, args, st);
    case 4: return launch_p1<4, 32, DENSE>(c, args, st);
    case 8: return launch_p1<8, 32, DENSE>(c, args, st);
    case 16: return launch_p1<16, 32, DENSE>(c, args, st);
    case 32: return launch_p1<32, 32, DENSE>(c, args, st);
    case 64: return launch_p1<64, 32, DENSE>(c, args, st);
    case 128: return launch_p1<128, 32, DENSE>(c, args, st);
  }
  return cudaErrorInvalidValue;
}

static cudaError_t launch_rowstage(Ctx* c, float2* y, const TemplateMeta* meta, int batch, int n_bands_all, int use_mask,
                                   cudaStream_t st) {
  k_rowstage<<<4 * c->n_sms, 256, 0, st>>>(y, ws_ptr<float2>(c, c->lay.tw_p2), meta, batch, c->prm.p,
                                                  c->log_n - kLogN2, n_bands_all, use_mask);
  c->launches++;
  return cudaGetLastError();
}

// The same values, band by band: row r of template I holds the 1024 bins of input row k1 of the narrow band l
// that owns compact row r (row_off[l] <= r < row_off[l+1]), with the bins outside the band set to 0, so that a
// band's rows are contiguous and need no masking by the consumer (k_fused stages them with one bulk copy).
__global__ void __launch_bounds__(256) k_correlate_bands(const TemplateMeta* __restrict__ meta, const float2* __restrict__ wq,
                                                         const double* __restrict__ u_tab, float2* __restrict__ qb, int p,
                                                         int rows_cap) {
  const TemplateMeta* m = meta + blockIdx.y;
  const int r = blockIdx.x;
  if (r >= m->row_off[p]) return;
  int l = 0;
  while (m->row_off[l + 1] <= r) ++l;
  const int e_lo = m->edges[l], e_hi = m->edges[l + 1];
  const int k1 = (e_lo >> kLogN2) + (r - m->row_off[l]);
  float2* out = qb + ((size_t)blockIdx.y * rows_cap + r) * kN2;
#pragma unroll
  for (int j = 0; j < 4; ++j) {
    const int k2 = threadIdx.x + 256 * j;
    const int k = (k1 << kLogN2) + k2;
    float2 v = make_float2(0.f, 0.f);
    if (k >= e_lo && k < e_hi) {
      const double u = u_tab[k];
      double t = fma(fma(fma(fma(m->c0, u * u, m->c2), u, m->c3), u, m->c4), u, -0.125);   // Psi0 / 2 pi, turns
      t -= rint(t);
      float sn, cs;
      sincospif(2.0f * (float)t, &sn, &cs);
      v = cmul(wq[k], make_float2(cs, sn));
    }
    out[k2] = v;
  }
}

cudaError_t launch_correlate_bands(Ctx* c, int first, int count, int parity, cudaStream_t st) {
  const int cap = qb_rows_cap(c);
  k_correlate_bands<<<dim3(c->n1 / 2 + c->prm.p + 1, count), 256, 0, st>>>(
      ws_ptr<TemplateMeta>(c, c->lay.meta) + first, wq_buf(c, c->front), ws_ptr<double>(c, c->lay.u_tab),
      ws_ptr<float2>(c, c->lay.qb) + (size_t)parity * c->lay.batch * cap * kN2, c->prm.p, cap);
  c->launches++;
  return cudaGetLastError();
}

cudaError_t launch_correlate(Ctx* c, int first, int count, int parity, cudaStream_t st, bool c_major) {
  const int half = (int)(c->n / 2);
  // only the bins some template of the batch owns: k_low .. the batch's largest k_high (host-side bank scalars)
  int kh = 0;
  for (int t = first; t < first + count; ++t) kh = c->h_meta[t].k_high > kh ? c->h_meta[t].k_high : kh;
  float2* q = ws_ptr<float2>(c, c->lay.q) + (size_t)parity * c->lay.batch * half;
  if (c_major) {
    const int row_first = c->k_low >> kLogN2, rows = ((kh - 1) >> kLogN2) - row_first + 1;
    if (rows <= 0) return cudaSuccess;
    k_correlate_cm<<<dim3(rows, count), 256, 0, st>>>(ws_ptr<TemplateMeta>(c, c->lay.meta) + first, wq_buf(c, c->front),
                                                      ws_ptr<double>(c, c->lay.u_tab), q, half, row_first);
    c->launches++;
    return cudaGetLastError();
  }
  const int k_first = c->k_low & ~255;
  const int blocks = (kh - k_first + 255) / 256;
  if (blocks <= 0) return cudaSuccess;
  k_correlate<<<dim3(blocks, count), 256, 0, st>>>(ws_ptr<TemplateMeta>(c, c->lay.meta) + first, wq_buf(c, c->front),
                                                  ws_ptr<double>(c, c->lay.u_tab), q, half, k_first);
  c->launches++;
  return cudaGetLastError();
}

// Pass 1 of one batch.  The narrow-band kernel (almost all of the work) runs on the context's stream; the
// low-volume kernels -- the generic kernel and the row stage for the wide bands, and the correlate kernel
// of the NEXT batch (next_count > 0) into the other half of the double-buffered Q -- run beside it on a
// high-priority side stream between a fork and a join event.  q_ready: this batch's Q was already produced
// by the previous call.
cudaError_t launch_pass1_filter(Ctx* c, int first, int count, int next_first, int next_count, int parity, bool q_ready) {
  P1Args args;
  args.meta = ws_ptr<TemplateMeta>(c, c->lay.meta) + first;
  args.wq = wq_buf(c, c->front);
  args.u_tab = ws_ptr<double>(c, c->lay.u_tab);
  args.tw_n1 = ws_ptr<float2>(c, c->lay.tw_n1);
  args.dense_in = nullptr;
  args.y = ws_ptr<float2>(c, c->lay.y);
  args.p = c->prm.p;
  args.log_n = c->log_n;
  args.n1 = c->n1;
  args.batch = count;
  args.slot_base = 0;
  args.first_template = 0;
  args.ja_per_cta = 1;
  args.ubuf = nullptr;
  args.vbuf = nullptr;
  args.tw_p2 = ws_ptr<float2>(c, c->lay.tw_p2);
  args.q = ws_ptr<float2>(c, c->lay.q) + (size_t)parity * c->lay.batch * (size_t)(c->n / 2);
  cudaError_t e;
  if (!q_ready) {
    e = launch_correlate(c, first, count, parity, c->stream);
    if (e == cudaSuccess && c->fused) e = launch_correlate_bands(c, first, count, parity, c->stream);
    if (e != cudaSuccess) return e;
    // (the side stream's correlates of an earlier call are complete: gwmf_triggers / any sync came in between,
    // or they were ordered before this call's work through the previous join)
  }
  // fork: everything enqueued so far on the main stream (this batch's Q, the previous batch's pass 2, which
  // read the band buffer) precedes the side work
  if ((e = cudaEventRecord(c->ev_fork, c->stream)) != cudaSuccess) return e;
  if ((e = cudaStreamWaitEvent(c->side, c->ev_fork, 0)) != cudaSuccess) return e;
  // which kernels have anything to do: host mirror of the wide-band masks (written by k_bank_setup; the caller has
  // waited for it once since the last bank setup, api.cu:ensure_mirror)
  const uint32_t full = c->prm.p >= 32 ? 0xFFFFFFFFu : ((1u << c->prm.p) - 1u);
  bool any_wide = false, any_narrow = false;
  for (int t = first; t < first + count; ++t) {
    any_wide |= c->h_masks[t] != 0u;
    any_narrow |= c->h_masks[t] != full;
  }
  if (any_narrow && !c->fused) {
    // narrow bands write the A layout directly
    e = launch_narrow(c, args, count);
    if (e != cudaSuccess) return e;
  }
  if (any_wide) {
    // wide bands (every band if n1 < 32): generic kernel in the plain layout, then the row stage in place
    e = dispatch_p1<false>(c, args, c->side);
    if (e != cudaSuccess) return e;
    e = launch_rowstage(c, args.y, args.meta, count, count * c->prm.p, 1, c->side);
    if (e != cudaSuccess) return e;
  }
  if (c->fused) {
    // the spill-free kernel only waits for the wide bands; the next batch's correlates then run beside it
    if ((e = cudaEventRecord(c->ev_join, c->side)) != cudaSuccess) return e;
    if (next_count > 0) {
      bool next_wide = false;
      for (int t = next_first; t < next_first + next_count; ++t) next_wide |= c->h_masks[t] != 0u;
      e = launch_correlate_bands(c, next_first, next_count, parity ^ 1, c->side);
      if (e == cudaSuccess && next_wide) e = launch_correlate(c, next_first, next_count, parity ^ 1, c->side);
      if (e != cudaSuccess) return e;
    }
    return cudaStreamWaitEvent(c->stream, c->ev_join, 0);
  }
  if (next_count > 0) {
    e = launch_correlate(c, next_first, next_count, parity ^ 1, c->side);
    if (e != cudaSuccess) return e;
  }
  if ((e = cudaEventRecord(c->ev_join, c->side)) != cudaSuccess) return e;
  return cudaStreamWaitEvent(c->stream, c->ev_join, 0);
}

cudaError_t launch_pass1_dense(Ctx* c, const float2* d_in, float2* d_mid, cudaStream_t st) {
  P1Args args;
  args.meta = nullptr;
  args.wq = nullptr;
  args.u_tab = nullptr;
  args.tw_n1 = ws_ptr<float2>(c, c->lay.tw_n1);
  args.tw_p2 = ws_ptr<float2>(c, c->lay.tw_p2);
  args.q = nullptr;
  args.dense_in = d_in;
  args.y = d_mid;
  args.p = 1;
  args.log_n = c->log_n;
  args.n1 = c->n1;
  args.batch = 1;
  args.slot_base = 0;
  args.first_template = 0;
  args.ja_per_cta = 1;
  args.ubuf = nullptr;
  args.vbuf = nullptr;
  return dispatch_p1<true>(c, args, st);
}

cudaError_t launch_rowstage_dense(Ctx* c, float2* d_mid, cudaStream_t st) { return launch_rowstage(c, d_mid, nullptr, 1, 1, 0, st); }

// ---- decimated path launchers ---------------------------------------------------------------------
static void fill_eff_args(Ctx* c, P1Args& args, int first, int count, int parity) {
  args.meta = ws_ptr<TemplateMeta>(c, c->lay.meta) + first;
  args.wq = wq_buf(c, c->front);
  args.u_tab = ws_ptr<double>(c, c->lay.u_tab);
  args.tw_n1 = ws_ptr<float2>(c, c->lay.tw_n1);
  args.tw_p2 = ws_ptr<float2>(c, c->lay.tw_p2);
  args.q = ws_ptr<float2>(c, c->lay.q) + (size_t)parity * c->lay.batch * (size_t)(c->n / 2);
  args.dense_in = nullptr;
  args.y = ws_ptr<float2>(c, c->lay.y);
  args.p = c->prm.p;
  args.log_n = c->log_n;
  args.n1 = c->n1;
  args.batch = count;
  args.slot_base = c->h_eff[first];
  args.first_template = first;
  args.ja_per_cta = 1;
  args.ubuf = ws_ptr<float2>(c, c->lay.ubuf) + (size_t)parity * c->lay.batch * kUCap;
  args.vbuf = ws_ptr<float2>(c, c->lay.vbuf);
}

// first pass of every effective band of the batch (needs Q and U+ of the batch; host mirror h_eff valid)
cudaError_t launch_pass1_eff(Ctx* c, int first, int count, int parity, cudaStream_t st) {
  P1Args args;
  fill_eff_args(c, args, first, count, parity);
  const int n_slots = c->h_eff[first + count] - c->h_eff[first];
  if (n_slots <= 0) return cudaSuccess;
  args.ja_per_cta = c->na >= kP1JaPerCta ? kP1JaPerCta : c->na;
  k_pass1_eff<<<dim3(kP1Groups * (c->na / args.ja_per_cta), n_slots), kP1Warps * 32, kP1WSmem, st>>>(args, ws_ptr<SlotDesc>(c, c->lay.slot_tab));
  c->launches++;
  return cudaGetLastError();
}

// the effective bands flagged in gen_mask (very many input rows): 32-point transform over the rounds, into vbuf
cudaError_t launch_prepass(Ctx* c, int first, int count, int parity, cudaStream_t st) {
  P1Args args;
  fill_eff_args(c, args, first, count, parity);
  const int n_slots = c->h_eff[first + count] - c->h_eff[first];
  if (n_slots <= 0) return cudaSuccess;
  int* list = ws_ptr<int>(c, c->lay.pp_jobs);
  k_pp_jobs<<<1, 256, 0, st>>>(ws_ptr<SlotDesc>(c, c->lay.slot_tab), args.slot_base, n_slots, list + 1, list);
  k_prepass<<<8 * c->n_sms, 256, 0, st>>>(args, ws_ptr<SlotDesc>(c, c->lay.slot_tab), ws_ptr<float2>(c, c->lay.vbuf), list + 1, list);
  c->launches += 2;
  return cudaGetLastError();
}

template <int NA, int NB>
static cudaError_t configure_p1_one() {
  cudaError_t e = cudaFuncSetAttribute(k_pass1<NA, NB, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)p1_smem<NA, NB>());
  if (e == cudaSuccess)
    e = cudaFuncSetAttribute(k_pass1<NA, NB, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)p1_smem<NA, NB>());
  return e;
}

// Opt-in to > 48 KB of dynamic shared memory for every pass-1 kernel, on the CURRENT device (called by gwmf_create
// for each context: the attribute is per device, not per process).
cudaError_t configure_pass1(int /*path*/) {
  cudaError_t e = cudaFuncSetAttribute(k_pass1_narrow, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)kNarrowSmem);
  if (e == cudaSuccess) e = cudaFuncSetAttribute(k_pass1_eff, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)kP1WSmem);
  if (e == cudaSuccess) e = configure_p1_one<1, 16>();
  if (e == cudaSuccess) e = configure_p1_one<1, 32>();
  if (e == cudaSuccess) e = configure_p1_one<2, 32>();
  if (e == cudaSuccess) e = configure_p1_one<4, 32>();
  if (e == cudaSuccess) e = configure_p1_one<8, 32>();
  if (e == cudaSuccess) e = configure_p1_one<16, 32>();
  if (e == cudaSuccess) e = configure_p1_one<32, 32>();
  if (e == cudaSuccess) e = configure_p1_one<64, 32>();
  if (e == cudaSuccess) e = configure_p1_one<128, 32>();
  return e;
}

}  // namespace gwmf
