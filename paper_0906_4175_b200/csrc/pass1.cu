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
  // decimated path (effective bands, gwmf_internal.cuh): y is indexed by slot = eff_prefix - slot_base + e
  int eff;                    // 0: y is indexed by tb * p + l (two-pass / spill-free paths)
  int slot_base;              // eff_prefix of the first template of the batch
  int first_template;         // bank index of the first template of the batch
  const float2* ubuf;         // [batch][kUCap] one-sided power spectra U+ (bandpower.cu)
};

// The effective bands of a batch whose bit is set in TemplateMeta::gen_mask, as (tb << 6 | e), ascending, identical
// in every CTA.  s_list: batch * kMaxBands ints, s_cnt: batch + 1 ints of shared memory.  Returns the list length.
__device__ inline int build_gen_list(const TemplateMeta* meta, int batch, int* s_list, int* s_cnt) {
  for (int t = threadIdx.x; t < batch; t += blockDim.x) s_cnt[t] = __popc(meta[t].gen_mask);
  __syncthreads();
  if (threadIdx.x == 0) {
    int run = 0;
    for (int t = 0; t < batch; ++t) { const int v = s_cnt[t]; s_cnt[t] = run; run += v; }
    s_cnt[batch] = run;
  }
  __syncthreads();
  for (int t = threadIdx.x; t < batch; t += blockDim.x) {
    unsigned m = meta[t].gen_mask;
    int o = s_cnt[t];
    while (m) { const int e = __ffs(m) - 1; m &= m - 1; s_list[o++] = (t << 6) | e; }
  }
  __syncthreads();
  return s_cnt[batch];
}

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
    n_list = a.eff ? build_gen_list(a.meta, a.batch, s_list, s_cnt) : build_wide_list(a.meta, a.batch, a.p, s_list, s_cnt);

  const int tid = threadIdx.x;
  const int x = tid >> 3, c = tid & 7;
  const unsigned nmask = (1u << a.log_n) - 1u;
  const int n1 = a.n1;
  const int n_items = n_list * TILES * G;

#pragma unroll 1
  for (int item = blockIdx.x; item < n_items; item += gridDim.x) {
    const int tile = item % TILES, r = (item / TILES) % G;
    int band_index = DENSE ? 0 : s_list[item / (TILES * G)];      // tb * p + l (eff: tb << 6 | e, replaced by the slot)
    const int k2 = tile * C + c;

    int e_lo, e_hi, tb_q = 0;
    if constexpr (DENSE) {
      e_lo = 0;
      e_hi = 1 << a.log_n;
    } else if (a.eff) {
      const int tb = band_index >> 6, e = band_index & 63;
      const TemplateMeta* m = a.meta + tb;
      const EffBand eb = eff_band(m, e);                // only class-D bands are ever generic: src = Q, no holes
      e_lo = eb.e_lo;
      e_hi = eb.e_hi;
      tb_q = tb;
      band_index = m->eff_prefix - a.slot_base + e;
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
      float2* out = a.y + ((size_t)band_index * n1 + (size_t)(G * m + r)) * kN2 + k2;
#pragma unroll
      for (int jb = 0; jb < NB; ++jb)
        out[(size_t)jb * NA * kN2] = cmul(v[brev<NB>(jb)], Bt[jb * C + c]);
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
                                                  int n_bands_all, int use_mask, int slot_base) {
  // use_mask: 0 = every band, 1 = the wide bands (wide_mask), 2 = the generic effective bands (gen_mask, decimated path)
  __shared__ int s_list[kMaxBatch * kMaxBands];
  __shared__ int s_cnt[kMaxBatch + 1];
  const int n_list = use_mask == 2 ? build_gen_list(meta, batch, s_list, s_cnt)
                   : use_mask ? build_wide_list(meta, batch, p, s_list, s_cnt) : n_bands_all;
  if (use_mask == 2) {                                   // (tb << 6 | e) -> slot
    for (int i = threadIdx.x; i < n_list; i += blockDim.x) {
      const int v = s_list[i];
      s_list[i] = meta[v >> 6].eff_prefix - slot_base + (v & 63);
    }
    __syncthreads();
  }
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
// of input rows.  Same CTA shape and phases as k_pass1_narrow; what is new is the sum over the input rows that share
// a residue b' = (k1 - row_lo) mod 32: with k1 = row_lo + b' + 32 t,
//     sum_t X[k_t] e^{2 pi i ja k_t/n} = e^{2 pi i ja k_0/n} sum_t X[k_t] g^t,  g = e^{2 pi i ja 32 * 1024/n} = e^{2 pi i ja/NA},
// evaluated by Horner's rule with the CTA-constant g: ceil(R/32) complex multiply-adds per (b', column), then the
// same 32-point transform over b'.  Bands of at most 16 rows keep the pruned variants.  Bins of class-D bands that
// lie inside the hull of Z ("holes": only with unusual spectra) are masked out.
// ---------------------------------------------------------------------------------------------------
struct EffSrc {
  const float2* src;      // spectrum indexed by absolute bin k (Q of the template, or U+ of the template)
  int e_lo, e_hi;
  int n_holes;            // Z only
  const int* holes;       // shared memory: [2h] = first bin of hole h, [2h+1] = one past its last bin
};

// Input of thread (column k2) from row k1, staged through shared memory by an 8-byte cp.async (LDGSTS): no
// register is tied up while the load is in flight, so a whole round of 32 rows is requested at once.  Rows strictly
// inside the band need no bin test: fr / lr are the first / last row whose bin in THIS column belongs to the band
// (the band's first and last row are only partly inside); a masked element is zero-filled (src-size 0).
template <bool HOLES>
__device__ __forceinline__ void eff_request(const EffSrc& es, float2* slot, int k1, int k2, int fr, int lr) {
  const int k = k1 * kN2 + k2;                  // k1 is negative for the lower half of a pair spectrum
  bool ok = k1 >= fr && k1 <= lr;
  if constexpr (HOLES) {
    for (int h = 0; h < es.n_holes; ++h) ok = ok && !(k >= es.holes[2 * h] && k < es.holes[2 * h + 1]);
  }
  const float2* src = es.src + (ok ? k : es.e_lo);                 // always a valid address
  asm volatile("cp.async.ca.shared.global [%0], [%1], 8, %2;" ::"r"((unsigned)__cvta_generic_to_shared(slot)), "l"(src),
               "r"(ok ? 8 : 0)
               : "memory");
}
__device__ __forceinline__ void cp_async_commit() { asm volatile("cp.async.commit_group;" ::: "memory"); }
__device__ __forceinline__ void cp_async_wait_all() { asm volatile("cp.async.wait_group 0;" ::: "memory"); }

// First round of requests of a thread (rows row_lo + i + 32 (T-1), i < RMAX), issued BEFORE the CTA builds its
// twiddle tables so that their latency overlaps that work.  stage: [32 rows][256 columns] aliasing the exchange tile;
// a thread only ever touches its own column of it.
template <int RMAX, bool HOLES>
__device__ __forceinline__ void eff_request_round(const EffSrc& es, float2* stage_col, int row0, int k2, int fr, int lr) {
#pragma unroll
  for (int i = 0; i < RMAX; ++i) eff_request<HOLES>(es, stage_col + i * 256, row0 + i, k2, fr, lr);
  cp_async_commit();
}

// Plain (register) load of the same element, for the round that is requested first of all, while the registers of
// the transform are still free.
template <bool HOLES>
__device__ __forceinline__ float2 eff_load(const EffSrc& es, int k1, int k2, int fr, int lr) {
  const int k = k1 * kN2 + k2;                  // k1 is negative for the lower half of a pair spectrum
  bool ok = k1 >= fr && k1 <= lr;
  if constexpr (HOLES) {
    for (int h = 0; h < es.n_holes; ++h) ok = ok && !(k >= es.holes[2 * h] && k < es.holes[2 * h + 1]);
  }
  float2 val = make_float2(0.f, 0.f);
  if (ok) val = __ldg(es.src + k);
  return val;
}

// Phase 1 of a CTA: thread (m, ci) owns column k2 and forms, for every residue b' = (k1 - row_lo) mod 32,
//     v[b'] = TW[b'] sum_t X[row_lo + b' + 32 t][k2] g^t        (Horner, g = e^{2 pi i ja/NA})
// then the 32-point transform over b', the T1 twiddle, and writes its column of the exchange tile.
// TW[i] = e^{2 pi i ja (row_lo + i)/n1} (shared, CTA constant).  The column part e^{2 pi i ja k2/n} of the twiddle is
// split off: its m part rides on the T1 table (built per CTA), its c part on the per-thread twiddle of phase 2.
// Latency: round t = 0 is loaded straight into the registers v[] at the very top (they are free until the transform),
// the last round t = T-1 (if T > 1) goes through cp.async into the staging area at the same time; both are in flight
// while the CTA builds its tables.  Only bands of more than 64 rows have further rounds, requested one after the other.
template <int RMAX, bool HOLES>
__device__ __forceinline__ void eff_phase1(const P1Args& a, const EffSrc& es, float2* __restrict__ T1, float2* __restrict__ TW,
                                           float2* __restrict__ tile, int ja, int cg) {
  const int tid = threadIdx.x;
  const unsigned nmask = (1u << a.log_n) - 1u;
  const int n1m = a.n1 - 1;
  const int row_lo = es.e_lo >> kLogN2, row_hi = (es.e_hi - 1) >> kLogN2;
  const int R = row_hi - row_lo + 1;
  const int T = (R + 31) >> 5;
  const int ci = tid & 7, m = tid >> 3;
  const int k2 = 32 * m + 8 * cg + ci;
  const int fr = row_lo + (k2 < (es.e_lo & (kN2 - 1)) ? 1 : 0);
  const int lr = row_hi - (k2 > ((es.e_hi - 1) & (kN2 - 1)) ? 1 : 0);
  float2* stage_col = tile + tid;               // [i][256]: column tid = m * 8 + ci of the staging area

  float2 v[32];
  const bool preload = RMAX < 32 || T <= 2;     // CTA-uniform
  if (preload) {
#pragma unroll
    for (int i = 0; i < RMAX; ++i) v[brev<32>(i)] = eff_load<HOLES>(es, row_lo + i, k2, fr, lr);        // round 0
  }
  if constexpr (RMAX == 32) {
    if (T > 1) eff_request_round<32, HOLES>(es, stage_col, row_lo + 32 * (T - 1), k2, fr, lr);          // round T-1
  }
  if (tid < 32) TW[tid] = a.tw_n1[(ja * (row_lo + tid)) & n1m];
  __syncthreads();                              // T1 (built by the caller before the slot was known) and TW are ready

  if constexpr (RMAX == 32) {
    if (T > 1) {
      const tw4 g = make_tw4(a.tw_n1[(ja * 32) & n1m]);                          // e^{2 pi i ja/NA}
      cp_async_wait_all();                                                       // round T-1 has landed (own column only)
      if (preload) {                                                             // T == 2: v = stage g + v
#pragma unroll
        for (int i = 0; i < 32; ++i) {
          const float2 hi = stage_col[i * 256], val = v[brev<32>(i)];
          v[brev<32>(i)] = unpk(fma2(pk(-hi.y, hi.x), g.yy, fma2(pk(hi), g.xx, pk(val))));
        }
      } else {                                                                   // more than 64 rows: round after round
#pragma unroll
        for (int i = 0; i < 32; ++i) v[brev<32>(i)] = stage_col[i * 256];
#pragma unroll 1
        for (int t = T - 2; t >= 0; --t) {
          eff_request_round<32, HOLES>(es, stage_col, row_lo + 32 * t, k2, fr, lr);
          cp_async_wait_all();
#pragma unroll
          for (int i = 0; i < 32; ++i) {
            const float2 val = stage_col[i * 256], w = v[brev<32>(i)];
            v[brev<32>(i)] = unpk(fma2(pk(-w.y, w.x), g.yy, fma2(pk(w), g.xx, pk(val))));   // v g + val
          }
        }
      }
    }
  }
#pragma unroll
  for (int i = 0; i < RMAX; ++i) v[brev<32>(i)] = cmul(v[brev<32>(i)], TW[i]);
  fft_dit<32, RMAX>(v);                     // inputs i >= RMAX are zero: leading stages pruned
  if constexpr (RMAX == 32) __syncthreads();   // every thread has consumed its staged inputs: the tile may be written
  const float4* __restrict__ t1 = reinterpret_cast<const float4*>(T1 + m * kT1Stride);
#pragma unroll
  for (int jb = 0; jb < 32; jb += 2) {
    const float4 w = t1[jb >> 1];
    tile[jb * kTileStride + m * 8 + ci] = cmul(v[jb], make_float2(w.x, w.y));
    tile[(jb + 1) * kTileStride + m * 8 + ci] = cmul(v[jb + 1], make_float2(w.z, w.w));
  }
}

template <bool HOLES>
__device__ __forceinline__ void eff_cta(const P1Args& a, const EffSrc& es, float2* tile, float2* T1, float2* TW, int ja, int cg) {
  const int R = ((es.e_hi - 1) >> kLogN2) - (es.e_lo >> kLogN2) + 1;
  if (R <= 4) eff_phase1<4, HOLES>(a, es, T1, TW, tile, ja, cg);
  else if (R <= 8) eff_phase1<8, HOLES>(a, es, T1, TW, tile, ja, cg);
  else if (R <= 16) eff_phase1<16, HOLES>(a, es, T1, TW, tile, ja, cg);
  else eff_phase1<32, HOLES>(a, es, T1, TW, tile, ja, cg);
}

__global__ void __launch_bounds__(256, 3) k_pass1_eff(P1Args a, const SlotDesc* __restrict__ slot_tab) {
  extern __shared__ __align__(128) float2 smem[];
  float2* tile = smem;                          // [32][kStageStride] (phase 1: stride kTileStride; before that: input staging)
  float2* T1 = smem + 32 * kStageStride;        // [32 m][kT1Stride]  e^{2 pi i (jb/1024 + 32 ja/n) m}
  __shared__ float2 TW[32];                     // e^{2 pi i ja (row_lo + i)/n1}
  __shared__ int s_holes[2 * kMaxBands];

  const int tid = threadIdx.x;
  const int na = a.n1 >> 5;
  const int cg = blockIdx.x & 3, ja = blockIdx.x >> 2;
  const int slot = blockIdx.y;                  // batch-relative
  const unsigned nmask = (1u << a.log_n) - 1u;

  const SlotDesc d = slot_tab[a.slot_base + slot];      // one 32-byte load, same address in every thread
  {
    // While the descriptor is on its way: T1 row m for jb = 4 ci .. 4 ci + 3 times this thread's m part of the column
    // twiddle, e^{2 pi i ja 32 m/n} (depends on ja only)
    const int ci = tid & 7, m = tid >> 3;
    const float2 Am = cis_frac(((unsigned)ja * 32u * (unsigned)m) & nmask, a.log_n);
    const float4* src4 = reinterpret_cast<const float4*>(a.tw_p2 + m * 32 + 4 * ci);
    const float4 w0 = __ldg(src4), w1 = __ldg(src4 + 1);
    float4* dst = reinterpret_cast<float4*>(T1 + m * kT1Stride + 4 * ci);
    const float2 p0 = cmul(make_float2(w0.x, w0.y), Am), p1 = cmul(make_float2(w0.z, w0.w), Am);
    const float2 p2 = cmul(make_float2(w1.x, w1.y), Am), p3 = cmul(make_float2(w1.z, w1.w), Am);
    dst[0] = make_float4(p0.x, p0.y, p1.x, p1.y);
    dst[1] = make_float4(p2.x, p2.y, p3.x, p3.y);
  }
  if (d.generic) return;                        // very many rows: k_pass1 (generic) + k_rowstage write this slot
  const int tb = d.t - a.first_template;

  EffSrc es;
  es.e_lo = d.e_lo;
  es.e_hi = d.e_hi;
  es.holes = s_holes;
  es.n_holes = d.n_holes;
  es.src = d.kind == kEffU    ? a.ubuf + (size_t)tb * kUCap
           : d.kind == kEffUP ? a.ubuf + (size_t)(tb + 1) * kUCap              // bin 0 of the pair spectrum; bins run negative
                              : a.q + (size_t)tb * (size_t)(1u << (a.log_n - 1));
  const int row_lo = es.e_lo >> kLogN2;

  if (d.n_holes > 0) {                          // rare: class-D bands inside the hull of Z
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
    eff_cta<true>(a, es, tile, T1, TW, ja, cg);
  } else {
    eff_cta<false>(a, es, tile, T1, TW, ja, cg);
  }
  __syncthreads();

  float2* out0 = a.y + ((size_t)slot * a.n1 + (size_t)ja) * kN2 + cg * 256;   // row jb adds jb * na * 1024
  const size_t row_stride = (size_t)na * kN2;
  // ---- phase 2: thread (jb = lane, ci = warp)
  {
    const int jb = tid & 31, cw = tid >> 5;
    const int c = 8 * cg + cw;
    // e^{2 pi i jb (c + 1024 b0)/32768} (rest of the column twiddle e^{2 pi i NA jb k2/n} and the rotation w_32^{jb b0})
    // times the c part of e^{2 pi i ja k2/n}: one angle, exact in integers mod n
    const unsigned num = ((unsigned)jb * (unsigned)(c + 1024 * (row_lo & 31)) * (unsigned)na + (unsigned)ja * (unsigned)c) & nmask;
    const tw4 S = make_tw4(cis_frac(num, a.log_n));
    float2 x[32];
#pragma unroll
    for (int mm = 0; mm < 32; ++mm) x[brev<32>(mm)] = cmul_tw(tile[jb * kTileStride + mm * 8 + cw], S);
    fft_dit<32>(x);                                   // over m -> jm
    __syncthreads();                                  // the tile has been read by everyone: reuse it as staging
    float4* st = reinterpret_cast<float4*>(tile + jb * kStageStride + cw * 32);
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
                                   cudaStream_t st, int slot_base = 0) {
  k_rowstage<<<4 * c->n_sms, 256, 0, st>>>(y, ws_ptr<float2>(c, c->lay.tw_p2), meta, batch, c->prm.p,
                                                  c->log_n - kLogN2, n_bands_all, use_mask, slot_base);
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

cudaError_t launch_correlate(Ctx* c, int first, int count, int parity, cudaStream_t st) {
  const int half = (int)(c->n / 2);
  // only the bins some template of the batch owns: k_low .. the batch's largest k_high (host-side bank scalars)
  int kh = 0;
  for (int t = first; t < first + count; ++t) kh = c->h_meta[t].k_high > kh ? c->h_meta[t].k_high : kh;
  const int k_first = c->k_low & ~255;
  const int blocks = (kh - k_first + 255) / 256;
  if (blocks <= 0) return cudaSuccess;
  k_correlate<<<dim3(blocks, count), 256, 0, st>>>(ws_ptr<TemplateMeta>(c, c->lay.meta) + first, wq_buf(c, c->front),
                                                  ws_ptr<double>(c, c->lay.u_tab),
                                                  ws_ptr<float2>(c, c->lay.q) + (size_t)parity * c->lay.batch * half, half,
                                                  k_first);
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
  args.eff = 0;
  args.slot_base = 0;
  args.first_template = 0;
  args.ubuf = nullptr;
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
  args.eff = 0;
  args.slot_base = 0;
  args.first_template = 0;
  args.ubuf = nullptr;
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
  args.eff = 1;
  args.slot_base = c->h_eff[first];
  args.first_template = first;
  args.ubuf = ws_ptr<float2>(c, c->lay.ubuf) + (size_t)parity * c->lay.batch * kUCap;
}

// first pass of every effective band of the batch (needs Q and U+ of the batch; host mirror h_eff valid)
cudaError_t launch_pass1_eff(Ctx* c, int first, int count, int parity, cudaStream_t st) {
  P1Args args;
  fill_eff_args(c, args, first, count, parity);
  const int n_slots = c->h_eff[first + count] - c->h_eff[first];
  if (n_slots <= 0) return cudaSuccess;
  k_pass1_eff<<<dim3(4 * c->na, n_slots), 256, kNarrowSmem, st>>>(args, ws_ptr<SlotDesc>(c, c->lay.slot_tab));
  c->launches++;
  return cudaGetLastError();
}

// the effective bands flagged in gen_mask: generic kernel (plain layout) + row stage, into their slots
cudaError_t launch_pass1_generic_eff(Ctx* c, int first, int count, int parity, cudaStream_t st) {
  P1Args args;
  fill_eff_args(c, args, first, count, parity);
  cudaError_t e = dispatch_p1<false>(c, args, st);
  if (e != cudaSuccess) return e;
  return launch_rowstage(c, args.y, args.meta, count, 0, 2, st, args.slot_base);
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
  if (e == cudaSuccess) e = cudaFuncSetAttribute(k_pass1_eff, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)kNarrowSmem);
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
