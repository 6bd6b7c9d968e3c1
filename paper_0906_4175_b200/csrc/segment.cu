// segment.cu -- per-context tables, per-segment preparation (step a0) and per-template sigma / band
// edges (step a1's reductions).  None of this is on the per-template hot path.
#include "gwmf_internal.cuh"

namespace gwmf {

// ---------------------------------------------------------------------------------------------------
// Tables that depend only on the parameters.
//   u_tab[k]  = f_k^(-1/3) (fp64), k = 0 .. n/2-1 (u_tab[0] = 0)
//   tw_n1[m]  = e^{2 pi i m / n1}, m = 0 .. n1-1        (pass-1 inter-stage twiddles)
//   tw_p2[jm][c] = e^{2 pi i jm c / 1024}, 32 x 32      (pass-2 inter-stage twiddles)
//   tw_l[t]   = e^{2 pi i t / 16384}                    (coarse-grid transforms of the decimated path)
// ---------------------------------------------------------------------------------------------------
__global__ void k_tables(double* __restrict__ u_tab, float2* __restrict__ tw_n1, float2* __restrict__ tw_p2,
                         float2* __restrict__ tw_l, int half_n, int n1, double df) {
  int i = blockIdx.x * blockDim.x + threadIdx.x;
  if (i < kLMax) {                      // tw_l[t] = e^{2 pi i t / kLMax}: coarse-grid transforms of bandpower.cu
    double s, c;
    sincospi(2.0 * (double)i / (double)kLMax, &s, &c);
    tw_l[i] = make_float2((float)c, (float)s);
  }
  if (i < half_n) u_tab[i] = (i == 0) ? 0.0 : rcbrt((double)i * df);
  if (i < n1) {
    double s, c;
    sincospi(2.0 * (double)i / (double)n1, &s, &c);
    tw_n1[i] = make_float2((float)c, (float)s);
  }
  if (i < 1024) {
    int jm = i >> 5, cc = i & 31;
    double s, c;
    sincospi(2.0 * (double)(jm * cc) / 1024.0, &s, &c);
    tw_p2[i] = make_float2((float)c, (float)s);
  }
}

cudaError_t launch_tables(Ctx* c) {
  int half = (int)(c->n / 2);
  int work = half > kLMax ? half : kLMax;
  k_tables<<<(work + 255) / 256, 256, 0, c->stream>>>(ws_ptr<double>(c, c->lay.u_tab),
                                                      ws_ptr<float2>(c, c->lay.tw_n1),
                                                      ws_ptr<float2>(c, c->lay.tw_p2), ws_ptr<float2>(c, c->lay.tw_l), half,
                                                      c->n1, c->df);
  c->launches++;
  return cudaGetLastError();
}

// ---------------------------------------------------------------------------------------------------
// Segment preparation.
// ---------------------------------------------------------------------------------------------------
__global__ void k_real_to_complex(const float* __restrict__ s, float2* __restrict__ x, int64_t n) {
  int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (i < n) x[i] = make_float2(s[i], 0.f);
}

// g[k] = f_k^(-7/3) / S_n[k] = u^7 / S_n[k] for k_low <= k < n/2, else 0 (integrand of Eq. 4).
// flags[0] is raised if S_n is not finite and positive inside the band.
__global__ void k_power_terms(const double* __restrict__ sn, const double* __restrict__ u_tab,
                              double* __restrict__ g, int* __restrict__ flags, int k_low, int half_n) {
  int k = blockIdx.x * blockDim.x + threadIdx.x;
  if (k >= half_n) return;
  double v = 0.0;
  if (k >= k_low) {
    double S = sn[k];
    if (!(S > 0.0) || isinf(S)) {
      atomicOr(flags, 1);
    } else {
      double u = u_tab[k], u2 = u * u, u4 = u2 * u2;
      v = u4 * u2 * u / S;
    }
  }
  g[k] = v;
}

// Inclusive fp64 prefix sum C[k] = sum_{k' <= k} g[k'] with a FIXED summation order (so that sigma and the band
// edges are bit-reproducible): the table is cut into 1024 contiguous chunks of L entries; a chunk is summed
// sequentially, the chunk totals are scanned sequentially, and every chunk is then re-summed from its offset.
// One warp per chunk: coalesced loads into shared memory, one lane walks the chunk (the dependent chain of L
// fp64 adds is ~2 us), coalesced stores.  (Once per segment; 4 MiB.)
constexpr int kPrefixChunks = 1024;

__global__ void __launch_bounds__(32) k_prefix_totals(const double* __restrict__ g, double* __restrict__ totals, int half_n, int L) {
  extern __shared__ double sh[];
  const int lo = blockIdx.x * L, hi = min(lo + L, half_n);
  for (int k = lo + threadIdx.x; k < hi; k += 32) sh[k - lo] = g[k];
  __syncwarp();
  if (threadIdx.x == 0) {
    double acc = 0.0;
    for (int k = 0; k < hi - lo; ++k) acc += sh[k];
    totals[blockIdx.x] = acc;
  }
}

__global__ void k_prefix_scan(double* __restrict__ totals) {      // exclusive, sequential
  double run = 0.0;
  for (int i = 0; i < kPrefixChunks; ++i) { const double v = totals[i]; totals[i] = run; run += v; }
}

__global__ void __launch_bounds__(32) k_prefix_write(const double* __restrict__ g, const double* __restrict__ offsets,
                                                     double* __restrict__ c_tab, int half_n, int L) {
  extern __shared__ double sh[];
  const int lo = blockIdx.x * L, hi = min(lo + L, half_n);
  for (int k = lo + threadIdx.x; k < hi; k += 32) sh[k - lo] = g[k];
  __syncwarp();
  if (threadIdx.x == 0) {
    double acc = offsets[blockIdx.x];
    for (int k = 0; k < hi - lo; ++k) { acc += sh[k]; sh[k] = acc; }
  }
  __syncwarp();
  for (int k = lo + threadIdx.x; k < hi; k += 32) c_tab[k] = sh[k - lo];
}

// wq[k] = (4/n) conj(Z[k]) f_k^(-7/6) / S_n[k] / sigma_ref for k_low <= k < n/2, else 0, where
// Z = sum_j s[j] e^{+2 pi i jk/n} (so conj(Z) is the ordinary forward DFT D[k] of the real segment,
// DESIGN.md reading 1) and sigma_ref = sqrt(4 df C[n/2-1]) keeps every later fp32 quantity O(rho)
// whatever the units of s and S_n.
__global__ void k_weighted_spectrum(const float2* __restrict__ Z, const double* __restrict__ sn,
                                    const double* __restrict__ u_tab, const double* __restrict__ c_tab,
                                    float2* __restrict__ wq, int k_low, int half_n, double four_over_n,
                                    double four_df) {
  int k = blockIdx.x * blockDim.x + threadIdx.x;
  if (k >= half_n) return;
  float2 out = make_float2(0.f, 0.f);
  if (k >= k_low) {
    double S = sn[k];
    if (S > 0.0 && !isinf(S)) {
      double sigma_ref = sqrt(four_df * c_tab[half_n - 1]);
      double u = u_tab[k];
      double amp = u * u * u * sqrt(u);                 // f^(-7/6)
      double w = four_over_n * amp / (S * sigma_ref);
      float2 z = Z[k];
      out = make_float2((float)(w * (double)z.x), (float)(-w * (double)z.y));
    }
  }
  wq[k] = out;
}

// Mean power of the segment in a template's band (reading 23): P[k] = sum_{k' <= k} |wq[k']|^2, the same
// fixed-order chunked fp64 prefix sum as C[k] with the terms formed on the fly.  By Parseval the mean over the n samples
// of sum_l |z_l|^2, in units of rho^2, is scale_rho2 * P[k_high - 1] for every template: 2 in noise alone, more when the
// data hold a loud signal in the band -- matched by this template or not.
__device__ __forceinline__ double wq_power(const float2* __restrict__ wq, int k) {
  const float2 v = wq[k];
  return (double)v.x * (double)v.x + (double)v.y * (double)v.y;
}

__global__ void __launch_bounds__(32) k_pw_totals(const float2* __restrict__ wq, double* __restrict__ totals, int half_n, int L) {
  extern __shared__ double sh[];
  const int lo = blockIdx.x * L, hi = min(lo + L, half_n);
  for (int k = lo + threadIdx.x; k < hi; k += 32) sh[k - lo] = wq_power(wq, k);
  __syncwarp();
  if (threadIdx.x == 0) {
    double acc = 0.0;
    for (int k = 0; k < hi - lo; ++k) acc += sh[k];
    totals[blockIdx.x] = acc;
  }
}

__global__ void __launch_bounds__(32) k_pw_write(const float2* __restrict__ wq, const double* __restrict__ offsets,
                                                 double* __restrict__ pw, int half_n, int L) {
  extern __shared__ double sh[];
  const int lo = blockIdx.x * L, hi = min(lo + L, half_n);
  for (int k = lo + threadIdx.x; k < hi; k += 32) sh[k - lo] = wq_power(wq, k);
  __syncwarp();
  if (threadIdx.x == 0) {
    double acc = offsets[blockIdx.x];
    for (int k = 0; k < hi - lo; ++k) { acc += sh[k]; sh[k] = acc; }
  }
  __syncwarp();
  for (int k = lo + threadIdx.x; k < hi; k += 32) pw[k] = sh[k - lo];
}

// The preparation is cut in three so that the part that depends only on the samples (the transform) can run on the
// upload stream while filters of the previous segment still use the PSD tables and the other wq buffer.
// Scratch (own region of the workspace, 3 n complex): X = the segment as complex input, mid, Z = its transform.
cudaError_t launch_segment_fft(Ctx* c, int buf, cudaStream_t st) {
  float2* X = ws_ptr<float2>(c, c->lay.prep);
  float2* mid = X + c->n;
  float2* Z = X + 2 * c->n;
  k_real_to_complex<<<(unsigned)((c->n + 255) / 256), 256, 0, st>>>(s_buf(c, buf), X, c->n);
  c->launches++;
  cudaError_t e = cudaGetLastError();
  if (e != cudaSuccess) return e;
  return launch_fft_dense(c, X, mid, Z, st);
}

cudaError_t launch_psd_tables(Ctx* c, cudaStream_t st) {
  const int half = (int)(c->n / 2);
  int* flags = ws_ptr<int>(c, c->lay.flags);
  cudaError_t e = cudaMemsetAsync(flags, 0, sizeof(int), st);
  if (e != cudaSuccess) return e;
  k_power_terms<<<(half + 255) / 256, 256, 0, st>>>(ws_ptr<double>(c, c->lay.sn), ws_ptr<double>(c, c->lay.u_tab),
                                                    ws_ptr<double>(c, c->lay.g_tab), flags, c->k_low, half);
  const int L = (half + kPrefixChunks - 1) / kPrefixChunks;
  const size_t sm = (size_t)L * sizeof(double);
  double* totals = ws_ptr<double>(c, c->lay.prefix_totals);
  k_prefix_totals<<<kPrefixChunks, 32, sm, st>>>(ws_ptr<double>(c, c->lay.g_tab), totals, half, L);
  k_prefix_scan<<<1, 1, 0, st>>>(totals);
  k_prefix_write<<<kPrefixChunks, 32, sm, st>>>(ws_ptr<double>(c, c->lay.g_tab), totals, ws_ptr<double>(c, c->lay.c_tab), half, L);
  c->launches += 4;
  return cudaGetLastError();
}

cudaError_t launch_weighted_spectrum(Ctx* c, int buf, cudaStream_t st) {
  const int half = (int)(c->n / 2);
  const float2* Z = ws_ptr<float2>(c, c->lay.prep) + 2 * c->n;
  k_weighted_spectrum<<<(half + 255) / 256, 256, 0, st>>>(Z, ws_ptr<double>(c, c->lay.sn), ws_ptr<double>(c, c->lay.u_tab),
                                                          ws_ptr<double>(c, c->lay.c_tab), wq_buf(c, buf), c->k_low, half,
                                                          4.0 / (double)c->n, 4.0 * c->df);
  c->launches++;
  cudaError_t e = cudaGetLastError();
  if (e != cudaSuccess) return e;
  // power table of this buffer's weighted spectrum (own chunk totals per buffer: loads of the two buffers may overlap)
  const int L = (half + kPrefixChunks - 1) / kPrefixChunks;
  const size_t sm = (size_t)L * sizeof(double);
  double* totals = ws_ptr<double>(c, c->lay.pw_totals) + (size_t)buf * kPrefixChunks;
  k_pw_totals<<<kPrefixChunks, 32, sm, st>>>(wq_buf(c, buf), totals, half, L);
  k_prefix_scan<<<1, 1, 0, st>>>(totals);
  k_pw_write<<<kPrefixChunks, 32, sm, st>>>(wq_buf(c, buf), totals, pw_buf(c, buf), half, L);
  c->launches += 3;
  return cudaGetLastError();
}

// ---------------------------------------------------------------------------------------------------
// sigma and band edges of every template (Eq. 4; equal-power bands):
//   sigma^2 = 4 df C[k_high-1];  e_0 = k_low;  e_l = 1 + min{k : C[k] >= (l/p) C[k_high-1]};  e_p = k_high.
// One thread per (template, edge); the edges are binary searches in the monotone fp64 table.
// ---------------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(256) k_bank_setup(TemplateMeta* __restrict__ meta, uint32_t* __restrict__ masks,
                                                    const double* __restrict__ c_tab, int n_templates, int p, int k_low,
                                                    int half_n, double four_df, int all_wide, int s_bins, int t_max,
                                                    int on_demand) {
  // thread (l = threadIdx.x, template = 8 blockIdx.x + threadIdx.y): one band edge each, then the wide-band mask
  __shared__ int s_edges[8][kMaxBands + 1];
  const int l = threadIdx.x, ty = threadIdx.y;
  const int t = blockIdx.x * 8 + ty;
  const bool live = t < n_templates;
  int k_high = 0;
  double total = 0.0;
  if (live) {
    k_high = meta[t].k_high;
    total = c_tab[k_high - 1];
    int e;
    if (l == 0) e = k_low;
    else if (l >= p) e = k_high;
    else {
      const double target = ((double)l / (double)p) * total;
      int lo = k_low, hi = k_high - 1;          // smallest k in [lo, hi] with C[k] >= target
      while (lo < hi) {
        const int mid = (lo + hi) >> 1;
        if (c_tab[mid] >= target) hi = mid; else lo = mid + 1;
      }
      e = lo + 1;
    }
    s_edges[ty][l] = e;
    if (l == 0) s_edges[ty][kMaxBands] = k_high;
  }
  __syncthreads();
  if (!live) return;
  // bands for the generic pass-1 kernel: more than 32 input rows (or every band when n1 < 32)
  bool wide = false;
  int rows = 0;
  if (l < p) {
    const int e_lo = s_edges[ty][l], e_hi = s_edges[ty][l + 1];
    rows = e_hi > e_lo ? ((e_hi - 1) >> kLogN2) - (e_lo >> kLogN2) + 1 : 0;
    wide = all_wide || rows > 32;
  }
  const unsigned mask = __ballot_sync(0xFFFFFFFFu, wide);
  // rows of the narrow bands in the band-separated spectrum: exclusive prefix sum over the bands
  int incl = wide ? 0 : rows;
#pragma unroll
  for (int d = 1; d < 32; d <<= 1) {
    const int v = __shfl_up_sync(0xFFFFFFFFu, incl, d);
    if (l >= d) incl += v;
  }
  meta[t].row_off[l + 1] = (uint16_t)incl;
  if (l == 0) { meta[t].row_off[0] = 0; meta[t].row_off[kMaxBands + 1] = 0; }
  meta[t].edges[l] = s_edges[ty][l];
  // ---- decimated path: classes and effective bands (gwmf_internal.cuh).  s_bins == 0 switches it off.
  {
    int bins = 0, e_lo = 0, e_hi = 0;
    if (l < p) { e_lo = s_edges[ty][l]; e_hi = s_edges[ty][l + 1]; bins = e_hi - e_lo; }
    bool is_s = s_bins > 0 && bins > 0 && bins <= s_bins;
    // Z and U cost two n-point transforms: decimate only if that is fewer than the narrow bands themselves (this
    // also keeps n_eff <= p, the size the band buffer is carved for)
    if (__popc(__ballot_sync(0xFFFFFFFFu, is_s)) <= 2) is_s = false;
    const bool is_d = bins > 0 && !is_s;
    const unsigned s_mask = __ballot_sync(0xFFFFFFFFu, is_s), d_mask = __ballot_sync(0xFFFFFFFFu, is_d);
    const int z_lo = __reduce_min_sync(0xFFFFFFFFu, is_s ? e_lo : 0x7FFFFFFF);
    const int z_hi = __reduce_max_sync(0xFFFFFFFFu, is_s ? e_hi : 0);
    const int u_hi = __reduce_max_sync(0xFFFFFFFFu, is_s ? bins : 0);
    const int base = s_mask ? 2 : 0;
    // generic kernel for class-D bands of more than 32 t_max input rows (the Horner sum of k_pass1_eff would be long)
    unsigned gen = 0u;
    if (is_d && rows > 32 * t_max) gen = 1u << (base + __popc(d_mask & ((1u << l) - 1u)));
    gen = __reduce_or_sync(0xFFFFFFFFu, gen);
    if (l == 0) {
      meta[t].s_mask = s_mask;
      meta[t].d_mask = d_mask;
      meta[t].gen_mask = gen;
      meta[t].n_eff = base + __popc(d_mask);
      meta[t].z_lo = s_mask ? z_lo : 0;
      meta[t].z_hi = z_hi;
      meta[t].u_hi = u_hi;
      meta[t].full_band = 0;
      meta[t].pair = 0;
      meta[t].up_hi = 0;
      if (on_demand) {                          // one transform over the whole template; chi^2 comes later, per event
        const int k0 = s_edges[ty][0];
        const int rows_all = ((k_high - 1) >> kLogN2) - (k0 >> kLogN2) + 1;
        meta[t].s_mask = 0;
        meta[t].d_mask = 0;
        meta[t].gen_mask = rows_all > 32 * t_max ? 1u : 0u;
        meta[t].n_eff = 1;
        meta[t].full_band = 1;
      }
    }
  }
  if (l == 0) {
    meta[t].edges[kMaxBands] = k_high;
    meta[t].sigma = sqrt(four_df * total);
    meta[t].scale_rho2 = (float)(c_tab[half_n - 1] / total);
    meta[t].wide_mask = mask;
    masks[t] = mask;
  }
}

// eff_prefix[t] = sum_{t' < t} n_eff[t'] (exclusive), total in eff_out[n_templates]; eff_out[n_templates + 1 + t] = 1 if
// template t has a generic effective band.  One block; sequential over chunks, fixed order.
__global__ void __launch_bounds__(1024) k_eff_scan(TemplateMeta* __restrict__ meta, int32_t* __restrict__ eff_out, int n_templates) {
  __shared__ int part[1024];
  const int t = threadIdx.x;
  const int L = (n_templates + 1023) / 1024;
  const int lo = min(t * L, n_templates), hi = min(lo + L, n_templates);
  int acc = 0;
  for (int i = lo; i < hi; ++i) acc += meta[i].n_eff;
  part[t] = acc;
  __syncthreads();
  if (t == 0) {
    int run = 0;
    for (int i = 0; i < 1024; ++i) { const int v = part[i]; part[i] = run; run += v; }
    eff_out[n_templates] = run;
  }
  __syncthreads();
  acc = part[t];
  for (int i = lo; i < hi; ++i) {
    meta[i].eff_prefix = acc;
    eff_out[i] = acc;
    eff_out[n_templates + 1 + i] = meta[i].gen_mask ? 1 : 0;
    acc += meta[i].n_eff;
  }
}

// Pairs (decimated path): templates 2i and 2i+1 share ONE transform for their two real series sum_l |z_l|^2 when
// both have narrow bands: the owner (2i) carries the band UP = U_A + i U_B, the guest loses its U band.  Pairs are
// fixed by the bank index, so a template's result does not depend on how the bank is cut into launches.
__global__ void k_pairing(TemplateMeta* __restrict__ meta, int n_templates) {
  const int t = 2 * (blockIdx.x * blockDim.x + threadIdx.x);
  if (t + 1 >= n_templates) return;
  TemplateMeta* a = meta + t;
  TemplateMeta* b = meta + t + 1;
  if (!a->s_mask || !b->s_mask || a->full_band || b->full_band) return;
  a->pair = 1;
  a->up_hi = a->u_hi > b->u_hi ? a->u_hi : b->u_hi;
  b->pair = 2;
  b->n_eff -= 1;
  b->gen_mask = (b->gen_mask >> 2) << 1;          // its class-D bands move from e >= 2 to e >= 1
}

// slot table of the whole bank: one thread per (template, effective band)
__global__ void __launch_bounds__(256) k_slot_table(const TemplateMeta* __restrict__ meta, SlotDesc* __restrict__ tab,
                                                    int n_templates) {
  const int t = blockIdx.x * 8 + (threadIdx.x >> 5), e = threadIdx.x & 31;
  if (t >= n_templates) return;
  const TemplateMeta* m = meta + t;
  if (e >= m->n_eff) return;
  const EffBand eb = eff_band(m, e);
  SlotDesc d;
  d.t = t;
  d.kind = eb.kind;
  d.e_lo = eb.e_lo;
  d.e_hi = eb.e_hi;
  d.n_holes = 0;
  if (eb.kind == kEffZ) {
    unsigned dm = m->d_mask;
    while (dm) {
      const int l = __ffs(dm) - 1;
      dm &= dm - 1;
      if (m->edges[l] >= eb.e_lo && m->edges[l + 1] <= eb.e_hi) ++d.n_holes;
    }
  }
  d.generic = (m->gen_mask >> e) & 1u;
  d.pad0 = d.pad1 = 0;
  tab[m->eff_prefix + e] = d;
}

cudaError_t launch_bank_setup(Ctx* c) {
  const bool decim = c->path == GWMF_PATH_DECIMATED;
  k_bank_setup<<<(c->n_templates + 7) / 8, dim3(32, 8), 0, c->stream>>>(
      ws_ptr<TemplateMeta>(c, c->lay.meta), ws_ptr<uint32_t>(c, c->lay.masks), ws_ptr<double>(c, c->lay.c_tab),
      c->n_templates, c->prm.p, c->k_low, (int)(c->n / 2), 4.0 * c->df, c->nb == 32 ? 0 : 1, decim ? c->s_bins : 0, c->t_max,
      c->prm.chisq_mode == GWMF_CHISQ_ON_DEMAND ? 1 : 0);
  c->launches++;
  cudaError_t e = cudaGetLastError();
  if (e != cudaSuccess) return e;
  c->mirror_ready = false;
  if (decim) {
    int32_t* d_eff = ws_ptr<int32_t>(c, c->lay.eff);
    k_pairing<<<(c->n_templates / 2 + 255) / 256 + 1, 256, 0, c->stream>>>(ws_ptr<TemplateMeta>(c, c->lay.meta), c->n_templates);
    c->launches++;
    k_eff_scan<<<1, 1024, 0, c->stream>>>(ws_ptr<TemplateMeta>(c, c->lay.meta), d_eff, c->n_templates);
    k_slot_table<<<(c->n_templates + 7) / 8, 256, 0, c->stream>>>(ws_ptr<TemplateMeta>(c, c->lay.meta),
                                                                    ws_ptr<SlotDesc>(c, c->lay.slot_tab), c->n_templates);
    c->launches += 2;
    if ((e = cudaGetLastError()) != cudaSuccess) return e;
    e = cudaMemcpyAsync(c->h_eff, d_eff, sizeof(int32_t) * (size_t)(2 * c->n_templates + 1), cudaMemcpyDeviceToHost, c->stream);
    if (e != cudaSuccess) return e;
  }
  // host mirror of the wide-band masks: lets gwmf_filter skip kernels that would find nothing to do
  e = cudaMemcpyAsync(c->h_masks, ws_ptr<uint32_t>(c, c->lay.masks), sizeof(uint32_t) * (size_t)c->n_templates,
                      cudaMemcpyDeviceToHost, c->stream);
  if (e != cudaSuccess) return e;
  return cudaEventRecord(c->ev_masks, c->stream);
}

}  // namespace gwmf
