// triggers.cu -- trigger-slot reset and ordered compaction (step a5's output side).
// Events leave the device sorted by (template, window): counts per template, an exclusive scan over
// templates, then each template writes its windows in order.  No atomics, so the order is fixed.
#include "gwmf_internal.cuh"

namespace gwmf {

__global__ void k_reset_slots(Slot* __restrict__ slots, size_t count) {
  size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (i < count) { slots[i].key = 0ull; slots[i].aux = 0ull; }
}

// one warp per template: lanes look at 32 consecutive windows at a time
__global__ void __launch_bounds__(256) k_count(const Slot* __restrict__ slots, int* __restrict__ counts, int n_templates,
                                               int n_windows) {
  const int t = blockIdx.x * 8 + (threadIdx.x >> 5), lane = threadIdx.x & 31;
  if (t >= n_templates) return;
  const Slot* s = slots + (size_t)t * n_windows;
  int c = 0;
  for (int w0 = 0; w0 < n_windows; w0 += 32) {
    const bool hit = (w0 + lane < n_windows) && s[w0 + lane].key != 0ull;
    c += __popc(__ballot_sync(0xFFFFFFFFu, hit));
  }
  if (lane == 0) counts[t] = c;
}

// offsets[t] = sum_{t' < t} counts[t'], offsets[n_templates] = total (as long long in offsets64[0])
__global__ void __launch_bounds__(1024) k_scan(const int* __restrict__ counts, long long* __restrict__ offsets,
                                               int n_templates) {
  __shared__ long long part[1024];
  int t = threadIdx.x;
  int L = (n_templates + 1023) / 1024;
  int lo = min(t * L, n_templates), hi = min(lo + L, n_templates);
  long long acc = 0;
  for (int i = lo; i < hi; ++i) acc += counts[i];
  part[t] = acc;
  __syncthreads();
  if (t == 0) {
    long long run = 0;
    for (int i = 0; i < 1024; ++i) { long long v = part[i]; part[i] = run; run += v; }
    offsets[n_templates] = run;
  }
  __syncthreads();
  acc = part[t];
  for (int i = lo; i < hi; ++i) { offsets[i] = acc; acc += counts[i]; }
}

// one warp per template; within a template events keep window order (ballot + prefix popcount)
__global__ void __launch_bounds__(256) k_emit(const Slot* __restrict__ slots, const long long* __restrict__ offsets,
                                              gwmf_trigger* __restrict__ out, long long capacity, int n_templates,
                                              int n_windows) {
  const int t = blockIdx.x * 8 + (threadIdx.x >> 5), lane = threadIdx.x & 31;
  if (t >= n_templates) return;
  const Slot* s = slots + (size_t)t * n_windows;
  long long o = offsets[t];
  for (int w0 = 0; w0 < n_windows; w0 += 32) {
    const int w = w0 + lane;
    Slot sl;
    sl.key = 0ull; sl.aux = 0ull;
    if (w < n_windows) sl = s[w];
    const bool hit = sl.key != 0ull;
    const unsigned b = __ballot_sync(0xFFFFFFFFu, hit);
    const long long pos = o + __popc(b & ((1u << lane) - 1u));
    if (hit && pos < capacity) {
      gwmf_trigger g;
      g.template_id = t;
      g.sample = (int32_t)(0xFFFFFFFFu - (unsigned)(sl.key & 0xFFFFFFFFull));
      g.rho = __uint_as_float((unsigned)(sl.key >> 32));
      g.chisq = __uint_as_float((unsigned)(sl.aux & 0xFFFFFFFFull));
      out[pos] = g;
    }
    o += __popc(b);
  }
}

// ---------------------------------------------------------------------------------------------------
// chi^2 from its definition at one sample j, Eq. 5 with
//     z_l[j] = sum_{k in band l} Q[k] e^{2 pi i jk/n},   Q[k] = wq[k] e^{i Psi0(f_k)}        (Eq. 1)
// by one CTA of 256 threads in one pass over the template's bins: the phasor exactly as in k_correlate (fp64 Horner,
// reduced to one turn), the Fourier factor from jk mod n (exact in integers), fp32 sums per thread and a fixed-order
// block reduction per band (bit-reproducible); the p band sums are then combined as Eq. 5 prints it,
// chi^2 = (p / sigma^2) sum_l |z_l - z/p|^2, in fp64 -- NOT as sum |z_l|^2 - |z|^2 / p, whose two terms are of size
// rho^2 and cancel to a few digits at a loud event.  Cost O(k_high - k_low) per sample against O(p n log n) per template.
// Two uses:
//   chi^2 on demand (gwmf_params::chisq_mode = GWMF_CHISQ_ON_DEMAND; reading 21): the filter
//     has left, per (template, window), the maximum of rho and its sample; chi^2 is evaluated there and nowhere else;
//   loud events and samples (reading 23): in the every-sample mode the transforms' epilogue forms chi^2 as the
//     fp32 difference above, good to about rho^2 * 5e-7; where rho > kRhoLoud it is replaced by this evaluation.
// The result is valid in thread 0.  Every thread of the CTA must call it (it synchronises).
// ---------------------------------------------------------------------------------------------------
constexpr float kRhoLoud = 48.0f;

__device__ float chisq_definition(unsigned j, const TemplateMeta* __restrict__ m, const int* s_edges, float2* red, float2* s_z,
                                  const float2* __restrict__ wq, const double* __restrict__ u_tab, int p, int log_n) {
  const unsigned nmask = (1u << log_n) - 1u;
  const float inv_n2 = 2.0f / (float)(1u << log_n);
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  const double c0 = m->c0, c2 = m->c2, c3 = m->c3, c4 = m->c4;
  for (int l = 0; l < p; ++l) {
    float ax = 0.f, ay = 0.f;
    for (int k = s_edges[l] + threadIdx.x; k < s_edges[l + 1]; k += 256) {
      const double u = u_tab[k];
      double ph = fma(fma(fma(fma(c0, u * u, c2), u, c3), u, c4), u, -0.125);   // Psi0 / 2 pi, turns
      ph -= rint(ph);
      // total angle in turns: Psi0/2pi + (jk mod n)/n, both in [-1/2, 1): one sincospif
      const float turns = 2.0f * (float)ph + (float)((j * (unsigned)k) & nmask) * inv_n2;
      float sn, cs;
      sincospif(turns, &sn, &cs);
      const float2 v = wq[k];
      ax = fmaf(v.x, cs, fmaf(-v.y, sn, ax));
      ay = fmaf(v.x, sn, fmaf(v.y, cs, ay));
    }
#pragma unroll
    for (int d = 16; d > 0; d >>= 1) {
      ax += __shfl_down_sync(0xFFFFFFFFu, ax, d);
      ay += __shfl_down_sync(0xFFFFFFFFu, ay, d);
    }
    if (lane == 0) red[warp] = make_float2(ax, ay);
    __syncthreads();
    if (threadIdx.x == 0) {
      float sx = 0.f, sy = 0.f;
      for (int i = 0; i < 8; ++i) { sx += red[i].x; sy += red[i].y; }
      s_z[l] = make_float2(sx, sy);
    }
    __syncthreads();
  }
  float chi = 0.f;
  if (threadIdx.x == 0) {
    double zx = 0.0, zy = 0.0;
    for (int l = 0; l < p; ++l) { zx += (double)s_z[l].x; zy += (double)s_z[l].y; }
    zx /= (double)p;
    zy /= (double)p;
    double acc = 0.0;
    for (int l = 0; l < p; ++l) {
      const double dx = (double)s_z[l].x - zx, dy = (double)s_z[l].y - zy;
      acc += dx * dx + dy * dy;
    }
    chi = (float)(acc * (double)p * (double)m->scale_rho2);                      // Eq. 5
  }
  __syncthreads();                                            // s_z, red are free again
  return chi;
}

// chi^2 on demand: one CTA per (window, template) slot, every event.
__global__ void __launch_bounds__(256) k_chisq_at(Slot* __restrict__ slots, const TemplateMeta* __restrict__ meta,
                                                  const float2* __restrict__ wq, const double* __restrict__ u_tab, int p,
                                                  int n_windows, int log_n) {
  __shared__ float2 red[8];
  __shared__ float2 s_z[kMaxBands];
  __shared__ int s_edges[kMaxBands + 1];
  const int t = blockIdx.y, w = blockIdx.x;
  Slot* sl = slots + (size_t)t * n_windows + w;
  const unsigned long long key = sl->key;
  if (key == 0ull) return;                                    // no event in this window (uniform over the CTA)
  const unsigned j = 0xFFFFFFFFu - (unsigned)(key & 0xFFFFFFFFull);
  const TemplateMeta* m = meta + t;
  if (threadIdx.x <= p) s_edges[threadIdx.x] = m->edges[threadIdx.x];
  __syncthreads();
  const float chi = chisq_definition(j, m, s_edges, red, s_z, wq, u_tab, p, log_n);
  if (threadIdx.x == 0) sl->aux = (unsigned long long)__float_as_uint(chi);
}

// Every-sample mode: the events the epilogue's fp32 chi^2 is not good enough for (reading 23).  One CTA per
// template walks the template's events in window order and re-evaluates
//   those with rho > kRhoLoud: the difference sum |z_l|^2 - |z|^2 / p has lost its digits there (about rho^2 * 5e-7);
//   all of them if the data are loud in the template's band, i.e. the mean over the segment of sum_l |z_l|^2 (from the
//   power table of the weighted spectrum, segment.cu) exceeds kMeanLoud = twice its value in noise: the fp32 error of
//   the transforms scales with that mean and then shows in chi^2 at EVERY sample (measured 3e-3 per unit of excess;
//   a signal of optimal SNR A adds about 20 A^2 / n, whichever template looks at it).
// Templates without such events -- nearly all, nearly always -- cost one coalesced read of their slots.
constexpr float kMeanLoud = 4.0f;
__device__ __forceinline__ bool band_is_loud(const TemplateMeta* __restrict__ m, const double* __restrict__ pw) {
  return (float)((double)m->scale_rho2 * pw[m->k_high - 1]) > kMeanLoud;
}

__global__ void __launch_bounds__(256) k_chisq_loud(Slot* __restrict__ slots, const TemplateMeta* __restrict__ meta,
                                                    const float2* __restrict__ wq, const double* __restrict__ pw,
                                                    const double* __restrict__ u_tab, int p, int n_windows, int log_n) {
  __shared__ float2 red[8];
  __shared__ float2 s_z[kMaxBands];
  __shared__ int s_edges[kMaxBands + 1];
  __shared__ float s_max[8];
  __shared__ unsigned long long s_key[256];
  const int t = blockIdx.x;
  Slot* sl = slots + (size_t)t * n_windows;
  const TemplateMeta* m = meta + t;
  const bool all = band_is_loud(m, pw);                       // uniform over the CTA
  float mx = 0.f;
  for (int w = threadIdx.x; w < n_windows; w += 256) mx = fmaxf(mx, __uint_as_float((unsigned)(sl[w].key >> 32)));   // empty slot: key 0 = rho 0
#pragma unroll
  for (int d = 16; d > 0; d >>= 1) mx = fmaxf(mx, __shfl_xor_sync(0xFFFFFFFFu, mx, d));
  if ((threadIdx.x & 31) == 0) s_max[threadIdx.x >> 5] = mx;
  if (threadIdx.x <= p) s_edges[threadIdx.x] = m->edges[threadIdx.x];
  __syncthreads();
  mx = s_max[0];
#pragma unroll
  for (int i = 1; i < 8; ++i) mx = fmaxf(mx, s_max[i]);
  if (!(mx > (all ? 0.f : kRhoLoud))) return;                 // nothing to do (uniform over the CTA)
  const float bound = all ? 0.f : kRhoLoud;
  for (int w0 = 0; w0 < n_windows; w0 += 256) {
    s_key[threadIdx.x] = w0 + threadIdx.x < n_windows ? sl[w0 + threadIdx.x].key : 0ull;
    __syncthreads();
    for (int i = 0; i < 256; ++i) {
      const unsigned long long key = s_key[i];                // uniform over the CTA
      if (key == 0ull || !(__uint_as_float((unsigned)(key >> 32)) > bound)) continue;
      const unsigned j = 0xFFFFFFFFu - (unsigned)(key & 0xFFFFFFFFull);
      const float chi = chisq_definition(j, m, s_edges, red, s_z, wq, u_tab, p, log_n);
      if (threadIdx.x == 0) sl[w0 + i].aux = (unsigned long long)__float_as_uint(chi);
    }
    __syncthreads();
  }
}

// Series output (gwmf_series), same rule: a CTA owns 256 consecutive samples and re-evaluates chi^2 at those whose rho
// exceeds kRhoLoud, or at all of them if the data are loud in the template's band.
__global__ void __launch_bounds__(256) k_chisq_series_loud(const float* __restrict__ series_rho, float* __restrict__ series_chi,
                                                           const TemplateMeta* __restrict__ m, const float2* __restrict__ wq,
                                                           const double* __restrict__ pw, const double* __restrict__ u_tab,
                                                           int p, int log_n) {
  __shared__ float2 red[8];
  __shared__ float2 s_z[kMaxBands];
  __shared__ int s_edges[kMaxBands + 1];
  __shared__ float s_rho[256];
  const float bound = band_is_loud(m, pw) ? -1.0f : kRhoLoud;
  const unsigned j0 = blockIdx.x * 256u;
  s_rho[threadIdx.x] = series_rho[j0 + threadIdx.x];
  if (threadIdx.x <= p) s_edges[threadIdx.x] = m->edges[threadIdx.x];
  __syncthreads();
  for (int i = 0; i < 256; ++i) {
    if (!(s_rho[i] > bound)) continue;                        // uniform over the CTA
    const float chi = chisq_definition(j0 + i, m, s_edges, red, s_z, wq, u_tab, p, log_n);
    if (threadIdx.x == 0) series_chi[j0 + i] = chi;
  }
}

// chi^2 of the events of templates [first, first + count): every event (loud_only = false: chi^2 on demand) or only
// those the every-sample mode re-evaluates (k_chisq_loud).
cudaError_t launch_chisq_at_events(Ctx* c, int first, int count, bool loud_only) {
  Slot* slots = ws_ptr<Slot>(c, c->lay.slots) + (size_t)first * c->n_windows;
  const TemplateMeta* meta = ws_ptr<TemplateMeta>(c, c->lay.meta) + first;
  if (loud_only) {
    if (count <= 0) return cudaSuccess;
    k_chisq_loud<<<count, 256, 0, c->stream>>>(slots, meta, wq_buf(c, c->front), pw_buf(c, c->front),
                                               ws_ptr<double>(c, c->lay.u_tab), c->prm.p, c->n_windows, c->log_n);
    c->launches++;
    return cudaGetLastError();
  }
  // the template index rides on gridDim.y (at most 65535): a longer range goes out in several launches
  constexpr int kMaxGridY = 65535;
  for (int done = 0; done < count; done += kMaxGridY) {
    const int cnt = count - done < kMaxGridY ? count - done : kMaxGridY;
    k_chisq_at<<<dim3(c->n_windows, cnt), 256, 0, c->stream>>>(
        slots + (size_t)done * c->n_windows, meta + done, wq_buf(c, c->front), ws_ptr<double>(c, c->lay.u_tab), c->prm.p,
        c->n_windows, c->log_n);
    c->launches++;
    const cudaError_t e = cudaGetLastError();
    if (e != cudaSuccess) return e;
  }
  return cudaSuccess;
}

cudaError_t launch_chisq_series_loud(Ctx* c, int template_id, const float* series_rho, float* series_chi) {
  k_chisq_series_loud<<<(unsigned)(c->n / 256), 256, 0, c->stream>>>(
      series_rho, series_chi, ws_ptr<TemplateMeta>(c, c->lay.meta) + template_id, wq_buf(c, c->front), pw_buf(c, c->front),
      ws_ptr<double>(c, c->lay.u_tab), c->prm.p, c->log_n);
  c->launches++;
  return cudaGetLastError();
}

cudaError_t launch_reset_slots(Ctx* c, int first, int count) {
  size_t n = (size_t)count * c->n_windows;
  if (n == 0) return cudaSuccess;
  k_reset_slots<<<(unsigned)((n + 255) / 256), 256, 0, c->stream>>>(
      ws_ptr<Slot>(c, c->lay.slots) + (size_t)first * c->n_windows, n);
  c->launches++;
  return cudaGetLastError();
}

cudaError_t launch_compact(Ctx* c) {
  const Slot* slots = ws_ptr<Slot>(c, c->lay.slots);
  int* counts = ws_ptr<int>(c, c->lay.counts);
  long long* offsets = ws_ptr<long long>(c, c->lay.offsets);
  int T = c->n_templates;
  long long cap = (long long)c->prm.max_templates * c->n_windows;
  k_count<<<(T + 7) / 8, 256, 0, c->stream>>>(slots, counts, T, c->n_windows);
  k_scan<<<1, 1024, 0, c->stream>>>(counts, offsets, T);
  k_emit<<<(T + 7) / 8, 256, 0, c->stream>>>(slots, offsets, ws_ptr<gwmf_trigger>(c, c->lay.trig_out), cap, T,
                                                 c->n_windows);
  c->launches += 3;
  return cudaGetLastError();
}

}  // namespace gwmf
