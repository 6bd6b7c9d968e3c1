// api.cu -- the C ABI of include/gwmf.h: argument checking, workspace carving, host-side bank
// arithmetic (phase coefficients, k_high) and the launch sequences.  No compute happens on the host
// beyond a handful of scalars per template.
#include <math.h>
#include <new>
#include <stdlib.h>
#include <string.h>
#include <vector>

#include "gwmf_internal.cuh"

using namespace gwmf;

namespace {

size_t align_up(size_t x, size_t a = 256) { return (x + a - 1) / a * a; }

bool is_pow2(int64_t v) { return v > 0 && (v & (v - 1)) == 0; }

bool params_ok(const gwmf_params* p) {
  if (!p) return false;
  if (!is_pow2(p->n) || p->n < (1 << 14) || p->n > (1 << 22)) return false;
  if (!(p->fs > 0.0) || !(p->f_low > 0.0) || !(p->f_low < 0.5 * p->fs)) return false;
  if (p->p < 1 || p->p > kMaxBands) return false;
  if (!is_pow2(p->window) || p->window > p->n) return false;
  if (p->max_templates < 1) return false;
  if (p->batch < 0 || p->batch > kMaxBatch) return false;
  if (!(p->rho_thresh >= 0.0)) return false;
  return true;
}

int default_batch(const gwmf_params* p) {
  // keep the band intermediate (batch * p * n * 8 B) near 2 GiB: many waves of CTAs per launch (kernel
  // tails and launch gaps amortised; measured 16 > 8 > 4 templates per launch at n = 2^20) while holding
  // about 1% of the 180 GB HBM
  double per = (double)p->p * (double)p->n * 8.0;
  int b = (int)(2147483648.0 / per);
  if (b < 1) b = 1;
  if (b > kMaxBatch) b = kMaxBatch;
  if (b > p->max_templates) b = p->max_templates;
  return b;
}

Layout make_layout(const gwmf_params* p) {
  Layout L;
  memset(&L, 0, sizeof(L));
  const size_t n = (size_t)p->n, half = n / 2;
  const size_t n1 = n / kN2;
  const size_t nw = n / (size_t)p->window;
  const size_t T = (size_t)p->max_templates;
  L.batch = p->batch > 0 ? p->batch : default_batch(p);
  if (L.batch > p->max_templates) L.batch = p->max_templates;
  size_t off = 0;
  auto take = [&](size_t bytes) { size_t o = off; off = align_up(off + bytes); return o; };
  L.u_tab = take(half * sizeof(double));
  L.c_tab = take(half * sizeof(double));
  L.g_tab = take(half * sizeof(double));
  L.sn = take((half + 1) * sizeof(double));
  L.wq = take(half * sizeof(float2));
  L.s_in = take(n * sizeof(float));
  L.tw_n1 = take(n1 * sizeof(float2));
  L.tw_p2 = take(1024 * sizeof(float2));
  L.meta = take(T * sizeof(TemplateMeta));
  L.slots = take(T * nw * sizeof(Slot));
  L.masks = take(T * sizeof(uint32_t));
  L.prefix_totals = take(1024 * sizeof(double));
  L.counts = take(T * sizeof(int));
  L.offsets = take((T + 1) * sizeof(long long));
  L.trig_out = take(T * nw * sizeof(gwmf_trigger));
  L.series_rho = take(n * sizeof(float));
  L.series_chi = take(n * sizeof(float));
  L.flags = take(256);
  L.q = take(2 * (size_t)L.batch * half * sizeof(float2));     // double-buffered across batches
  L.qb = take(2 * (size_t)L.batch * (n1 / 2 + kMaxBands + 2) * kN2 * sizeof(float2));   // band-separated copy (k_fused)
  size_t yb = (size_t)L.batch * (size_t)p->p * n * sizeof(float2);
  if (yb < 3 * n * sizeof(float2)) yb = 3 * n * sizeof(float2);   // the dense transform needs in/mid/out
  L.y_bytes = yb;
  L.y = take(yb);
  L.total = off;
  return L;
}

int fail_cuda(Ctx* c, cudaError_t e) {
  c->cuda_err = cudaGetErrorString(e);
  return GWMF_E_CUDA;
}

#define CU(call)                                       \
  do {                                                 \
    cudaError_t e__ = (call);                          \
    if (e__ != cudaSuccess) return fail_cuda(c, e__);  \
  } while (0)

// Host-side scalars of template I = (m1, m2) (phase of BASELINE.json:configs[0]):
// phase coefficients in turns for u = f^(-1/3), and the first bin above the template.
int fill_template(const Ctx* c, const gwmf_mass_pair& mp, TemplateMeta* t) {
  if (!(mp.m1 > 0.0) || !(mp.m2 > 0.0) || !isfinite(mp.m1) || !isfinite(mp.m2)) return GWMF_E_ARG;
  const double pi = 3.14159265358979323846;
  const double mt = (mp.m1 + mp.m2) * GWMF_T_SUN;
  const double eta = mp.m1 * mp.m2 / ((mp.m1 + mp.m2) * (mp.m1 + mp.m2));
  const double f_isco = 1.0 / (pow(6.0, 1.5) * pi * mt);
  const double f_cut = fmin(f_isco, 0.5 * c->prm.fs);
  long kh = (long)ceil(f_cut / c->df);
  if (kh > c->n / 2) kh = (long)(c->n / 2);
  if (kh <= c->k_low) return GWMF_E_EMPTY_TEMPLATE;
  // v = kappa / u, kappa = (pi M)^(1/3):  Psi0 = -pi/4 + 3/(128 eta) [v^-5 + a2 v^-3 + a3 v^-2 + a4 v^-1]
  const double kappa = cbrt(pi * mt);
  const double lead = 3.0 / (128.0 * eta) / (2.0 * pi);          // in turns
  const double a2 = 3715.0 / 756.0 + 55.0 * eta / 9.0;
  const double a3 = -16.0 * pi;
  const double a4 = 15293365.0 / 508032.0 + 27145.0 * eta / 504.0 + 3085.0 * eta * eta / 72.0;
  memset(t, 0, sizeof(*t));
  t->c0 = lead / pow(kappa, 5.0);
  t->c2 = lead * a2 / pow(kappa, 3.0);
  t->c3 = lead * a3 / (kappa * kappa);
  t->c4 = lead * a4 / kappa;
  t->k_high = (int32_t)kh;
  return GWMF_OK;
}

}  // namespace

extern "C" {

size_t gwmf_workspace_bytes(const gwmf_params* params) {
  if (!params_ok(params)) return 0;
  return make_layout(params).total;
}

int gwmf_create(const gwmf_params* params, void* d_workspace, size_t workspace_bytes, void* cuda_stream,
                gwmf_ctx** out) {
  if (!out) return GWMF_E_ARG;
  *out = nullptr;
  if (!params_ok(params) || !d_workspace) return GWMF_E_ARG;
  if (((uintptr_t)d_workspace & 255u) != 0) return GWMF_E_ARG;
  Layout L = make_layout(params);
  if (workspace_bytes < L.total) return GWMF_E_WORKSPACE;
  int dev = 0;
  cudaDeviceProp prop;
  if (cudaGetDevice(&dev) != cudaSuccess || cudaGetDeviceProperties(&prop, dev) != cudaSuccess) return GWMF_E_CUDA;
  if (prop.major < 10) return GWMF_E_CUDA;       // no fallback: sm_100 only
  Ctx* c = new (std::nothrow) Ctx();
  if (!c) return GWMF_E_ARG;
  c->prm = *params;
  c->n = params->n;
  c->log_n = 0;
  while ((1ll << c->log_n) < c->n) ++c->log_n;
  c->n1 = (int)(c->n / kN2);
  c->nb = c->n1 >= 32 ? 32 : c->n1;
  c->na = c->n1 / c->nb;
  c->df = params->fs / (double)params->n;
  c->k_low = (int)ceil(params->f_low / c->df);
  c->n_windows = (int)(c->n / params->window);
  c->n_sms = prop.multiProcessorCount;
  c->lay = L;
  c->ws = (char*)d_workspace;
  c->stream = (cudaStream_t)cuda_stream;
  c->n_templates = 0;
  c->have_bank = c->have_segment = false;
  {
    // path selection: the spill-free kernel wins while bands stay a few rows wide (n <= 2^20: measured +8..11 %
    // at n = 2^18 and 2^20, -18 % at 2^22); GWMF_FUSED=0/1 forces the two-pass / the spill-free path
    const char* f = getenv("GWMF_FUSED");
    if (f && (f[0] == '0' || f[0] == '1')) c->fused = f[0] == '1';
    else c->fused = params->n <= (1 << 20) && params->n >= (1 << 15);
  }
  c->launches = 0;
  c->h_meta = nullptr;
  c->h_masks = nullptr;
  c->side = nullptr;
  c->ev_fork = c->ev_join = c->ev_masks = nullptr;
  {
    int lo = 0, hi = 0;
    cudaDeviceGetStreamPriorityRange(&lo, &hi);
    if (cudaStreamCreateWithPriority(&c->side, cudaStreamNonBlocking, hi) != cudaSuccess ||
        cudaEventCreateWithFlags(&c->ev_fork, cudaEventDisableTiming) != cudaSuccess ||
        cudaEventCreateWithFlags(&c->ev_join, cudaEventDisableTiming) != cudaSuccess ||
        cudaEventCreateWithFlags(&c->ev_masks, cudaEventDisableTiming) != cudaSuccess ||
        cudaMallocHost((void**)&c->h_masks, sizeof(uint32_t) * (size_t)params->max_templates) != cudaSuccess) {
      if (c->side) cudaStreamDestroy(c->side);
      if (c->ev_fork) cudaEventDestroy(c->ev_fork);
      if (c->ev_join) cudaEventDestroy(c->ev_join);
      if (c->ev_masks) cudaEventDestroy(c->ev_masks);
      delete c;
      return GWMF_E_CUDA;
    }
  }
  if (cudaMallocHost((void**)&c->h_meta, sizeof(TemplateMeta) * (size_t)params->max_templates) != cudaSuccess) {
    c->h_meta = nullptr;
    gwmf_destroy(reinterpret_cast<gwmf_ctx*>(c));
    return GWMF_E_CUDA;
  }
  cudaError_t e = launch_tables(c);
  if (e == cudaSuccess) e = launch_reset_slots(c, 0, params->max_templates);
  if (e != cudaSuccess) {
    gwmf_destroy(reinterpret_cast<gwmf_ctx*>(c));
    return GWMF_E_CUDA;
  }
  *out = reinterpret_cast<gwmf_ctx*>(c);
  return GWMF_OK;
}

void gwmf_destroy(gwmf_ctx* ctx) {
  if (!ctx) return;
  Ctx* c = reinterpret_cast<Ctx*>(ctx);
  cudaStreamSynchronize(c->stream);
  if (c->side) { cudaStreamSynchronize(c->side); cudaStreamDestroy(c->side); }
  if (c->ev_fork) cudaEventDestroy(c->ev_fork);
  if (c->ev_join) cudaEventDestroy(c->ev_join);
  if (c->ev_masks) cudaEventDestroy(c->ev_masks);
  if (c->h_masks) cudaFreeHost(c->h_masks);
  if (c->h_meta) cudaFreeHost(c->h_meta);
  delete c;
}

int gwmf_make_bank(gwmf_ctx* ctx, const gwmf_mass_pair* host_masses, int32_t n_templates) {
  if (!ctx || !host_masses) return GWMF_E_ARG;
  Ctx* c = reinterpret_cast<Ctx*>(ctx);
  if (n_templates < 1 || n_templates > c->prm.max_templates) return GWMF_E_ARG;
  CU(cudaStreamSynchronize(c->stream));            // h_meta may still be in flight from a previous call
  for (int t = 0; t < n_templates; ++t) {
    int rc = fill_template(c, host_masses[t], &c->h_meta[t]);
    if (rc != GWMF_OK) return rc;
  }
  CU(cudaMemcpyAsync(ws_ptr<TemplateMeta>(c, c->lay.meta), c->h_meta, sizeof(TemplateMeta) * (size_t)n_templates,
                     cudaMemcpyHostToDevice, c->stream));
  c->n_templates = n_templates;
  c->have_bank = true;
  CU(launch_reset_slots(c, 0, c->prm.max_templates));
  if (c->have_segment) CU(launch_bank_setup(c));
  return GWMF_OK;
}

int gwmf_load_segment(gwmf_ctx* ctx, const float* s, const double* Sn) {
  if (!ctx || !s || !Sn) return GWMF_E_ARG;
  Ctx* c = reinterpret_cast<Ctx*>(ctx);
  CU(cudaMemcpyAsync(ws_ptr<float>(c, c->lay.s_in), s, sizeof(float) * (size_t)c->n, cudaMemcpyDefault, c->stream));
  CU(cudaMemcpyAsync(ws_ptr<double>(c, c->lay.sn), Sn, sizeof(double) * (size_t)(c->n / 2 + 1), cudaMemcpyDefault,
                     c->stream));
  // pinned host sources are copied truly asynchronously: wait so that the caller may free them
  cudaPointerAttributes at_s, at_p;
  bool dev_s = cudaPointerGetAttributes(&at_s, s) == cudaSuccess && at_s.type == cudaMemoryTypeDevice;
  bool dev_p = cudaPointerGetAttributes(&at_p, Sn) == cudaSuccess && at_p.type == cudaMemoryTypeDevice;
  cudaGetLastError();
  if (!dev_s || !dev_p) CU(cudaStreamSynchronize(c->stream));
  CU(launch_segment_prepare(c));
  c->have_segment = true;
  CU(launch_reset_slots(c, 0, c->prm.max_templates));
  if (c->have_bank) CU(launch_bank_setup(c));
  return GWMF_OK;
}

int gwmf_filter(gwmf_ctx* ctx, int32_t first_template, int32_t n_templates) {
  if (!ctx) return GWMF_E_ARG;
  Ctx* c = reinterpret_cast<Ctx*>(ctx);
  if (!c->have_bank || !c->have_segment) return GWMF_E_STATE;
  if (first_template < 0 || n_templates < 0 || first_template + n_templates > c->n_templates) return GWMF_E_ARG;
  if (n_templates == 0) return GWMF_OK;
  CU(launch_reset_slots(c, first_template, n_templates));
  int parity = 0;
  for (int done = 0; done < n_templates; done += c->lay.batch, parity ^= 1) {
    const int cnt = n_templates - done < c->lay.batch ? n_templates - done : c->lay.batch;
    const int rest = n_templates - done - cnt;
    const int next = rest < c->lay.batch ? rest : c->lay.batch;
    CU(launch_pass1_filter(c, first_template + done, cnt, first_template + done + cnt, next, parity, done > 0));
    if (c->fused) CU(launch_fused_filter(c, first_template + done, cnt, parity, true, nullptr, nullptr));
    else CU(launch_pass2_filter(c, first_template + done, cnt, true, nullptr, nullptr));
  }
  return GWMF_OK;
}

int gwmf_filter_timed(gwmf_ctx* ctx, int32_t first_template, int32_t n_templates, double* host_ms,
                      int32_t* host_launches) {
  if (!ctx || !host_ms || !host_launches) return GWMF_E_ARG;
  Ctx* c = reinterpret_cast<Ctx*>(ctx);
  if (!c->have_bank || !c->have_segment) return GWMF_E_STATE;
  if (first_template < 0 || n_templates < 1 || first_template + n_templates > c->n_templates) return GWMF_E_ARG;
  const int nb = (n_templates + c->lay.batch - 1) / c->lay.batch;
  std::vector<cudaEvent_t> ev((size_t)nb * 3);
  for (auto& e : ev) CU(cudaEventCreate(&e));
  CU(launch_reset_slots(c, first_template, n_templates));
  for (int b = 0; b < nb; ++b) {
    int done = b * c->lay.batch;
    int cnt = n_templates - done < c->lay.batch ? n_templates - done : c->lay.batch;
    const int rest = n_templates - done - cnt;
    const int next = rest < c->lay.batch ? rest : c->lay.batch;
    CU(cudaEventRecord(ev[3 * b], c->stream));
    CU(launch_pass1_filter(c, first_template + done, cnt, first_template + done + cnt, next, b & 1, b > 0));
    CU(cudaEventRecord(ev[3 * b + 1], c->stream));
    if (c->fused) CU(launch_fused_filter(c, first_template + done, cnt, b & 1, true, nullptr, nullptr));
    else CU(launch_pass2_filter(c, first_template + done, cnt, true, nullptr, nullptr));
    CU(cudaEventRecord(ev[3 * b + 2], c->stream));
  }
  CU(cudaStreamSynchronize(c->stream));
  host_ms[0] = host_ms[1] = 0.0;
  for (int b = 0; b < nb; ++b) {
    float m1 = 0.f, m2 = 0.f;
    CU(cudaEventElapsedTime(&m1, ev[3 * b], ev[3 * b + 1]));
    CU(cudaEventElapsedTime(&m2, ev[3 * b + 1], ev[3 * b + 2]));
    host_ms[0] += m1;
    host_ms[1] += m2;
  }
  host_launches[0] = host_launches[1] = nb;
  for (auto& e : ev) cudaEventDestroy(e);
  return GWMF_OK;
}

static int check_flags(Ctx* c) {
  int flag = 0;
  cudaError_t e = cudaMemcpyAsync(&flag, ws_ptr<int>(c, c->lay.flags), sizeof(int), cudaMemcpyDeviceToHost, c->stream);
  if (e == cudaSuccess) e = cudaStreamSynchronize(c->stream);
  if (e != cudaSuccess) return fail_cuda(c, e);
  return flag ? GWMF_E_ARG : GWMF_OK;
}

int gwmf_triggers(gwmf_ctx* ctx, gwmf_trigger* host_out, int64_t capacity, int64_t* n_out) {
  if (!ctx || !n_out || capacity < 0 || (capacity > 0 && !host_out)) return GWMF_E_ARG;
  Ctx* c = reinterpret_cast<Ctx*>(ctx);
  *n_out = 0;
  if (!c->have_bank || !c->have_segment) return GWMF_E_STATE;
  // compaction first, then ONE synchronisation for the input-check flag and the event count
  CU(launch_compact(c));
  int flag = 0;
  long long total = 0;
  CU(cudaMemcpyAsync(&flag, ws_ptr<int>(c, c->lay.flags), sizeof(int), cudaMemcpyDeviceToHost, c->stream));
  CU(cudaMemcpyAsync(&total, ws_ptr<long long>(c, c->lay.offsets) + c->n_templates, sizeof(long long),
                     cudaMemcpyDeviceToHost, c->stream));
  CU(cudaStreamSynchronize(c->stream));
  if (flag) return GWMF_E_ARG;
  *n_out = total;
  long long take = total < capacity ? total : capacity;
  if (take > 0) {
    CU(cudaMemcpyAsync(host_out, ws_ptr<gwmf_trigger>(c, c->lay.trig_out), sizeof(gwmf_trigger) * (size_t)take,
                       cudaMemcpyDeviceToHost, c->stream));
    CU(cudaStreamSynchronize(c->stream));
  }
  return total > capacity ? GWMF_E_CAPACITY : GWMF_OK;
}

static int fetch_meta(Ctx* c, std::vector<TemplateMeta>& v) {
  if (!c->have_bank || !c->have_segment) return GWMF_E_STATE;
  int rc = check_flags(c);
  if (rc != GWMF_OK) return rc;
  v.resize((size_t)c->n_templates);
  CU(cudaMemcpyAsync(v.data(), ws_ptr<TemplateMeta>(c, c->lay.meta), sizeof(TemplateMeta) * v.size(),
                     cudaMemcpyDeviceToHost, c->stream));
  CU(cudaStreamSynchronize(c->stream));
  return GWMF_OK;
}

int gwmf_sigma(gwmf_ctx* ctx, double* host_sigma) {
  if (!ctx || !host_sigma) return GWMF_E_ARG;
  Ctx* c = reinterpret_cast<Ctx*>(ctx);
  std::vector<TemplateMeta> v;
  int rc = fetch_meta(c, v);
  if (rc != GWMF_OK) return rc;
  for (size_t t = 0; t < v.size(); ++t) host_sigma[t] = v[t].sigma;
  return GWMF_OK;
}

int gwmf_band_edges(gwmf_ctx* ctx, int32_t* host_edges) {
  if (!ctx || !host_edges) return GWMF_E_ARG;
  Ctx* c = reinterpret_cast<Ctx*>(ctx);
  std::vector<TemplateMeta> v;
  int rc = fetch_meta(c, v);
  if (rc != GWMF_OK) return rc;
  const int p = c->prm.p;
  for (size_t t = 0; t < v.size(); ++t)
    for (int l = 0; l <= p; ++l) host_edges[t * (size_t)(p + 1) + l] = v[t].edges[l];
  return GWMF_OK;
}

int gwmf_series(gwmf_ctx* ctx, int32_t template_id, float* host_rho, float* host_chisq) {
  if (!ctx) return GWMF_E_ARG;
  Ctx* c = reinterpret_cast<Ctx*>(ctx);
  if (!c->have_bank || !c->have_segment) return GWMF_E_STATE;
  if (template_id < 0 || template_id >= c->n_templates) return GWMF_E_ARG;
  int rc = check_flags(c);
  if (rc != GWMF_OK) return rc;
  float* d_rho = ws_ptr<float>(c, c->lay.series_rho);
  float* d_chi = ws_ptr<float>(c, c->lay.series_chi);
  CU(launch_pass1_filter(c, template_id, 1, 0, 0, 0, false));
  if (c->fused) CU(launch_fused_filter(c, template_id, 1, 0, false, d_rho, d_chi));
  else CU(launch_pass2_filter(c, template_id, 1, false, d_rho, d_chi));
  if (host_rho)
    CU(cudaMemcpyAsync(host_rho, d_rho, sizeof(float) * (size_t)c->n, cudaMemcpyDeviceToHost, c->stream));
  if (host_chisq)
    CU(cudaMemcpyAsync(host_chisq, d_chi, sizeof(float) * (size_t)c->n, cudaMemcpyDeviceToHost, c->stream));
  CU(cudaStreamSynchronize(c->stream));
  return GWMF_OK;
}

int gwmf_correlate(gwmf_ctx* ctx, int32_t template_id, float* host_q) {
  if (!ctx || !host_q) return GWMF_E_ARG;
  Ctx* c = reinterpret_cast<Ctx*>(ctx);
  if (!c->have_bank || !c->have_segment) return GWMF_E_STATE;
  if (template_id < 0 || template_id >= c->n_templates) return GWMF_E_ARG;
  int rc = check_flags(c);
  if (rc != GWMF_OK) return rc;
  const size_t half = (size_t)(c->n / 2);
  float2* d_q = ws_ptr<float2>(c, c->lay.q);
  CU(cudaMemsetAsync(d_q, 0, half * sizeof(float2), c->stream));      // bins outside [k_low, k_high) are not written
  CU(launch_correlate(c, template_id, 1, 0, c->stream));
  CU(cudaMemcpyAsync(host_q, d_q, half * sizeof(float2), cudaMemcpyDeviceToHost, c->stream));
  CU(cudaStreamSynchronize(c->stream));
  return GWMF_OK;
}

int gwmf_fft_inverse(gwmf_ctx* ctx, const float* d_in, float* d_out) {
  if (!ctx || !d_in || !d_out || d_in == d_out) return GWMF_E_ARG;
  Ctx* c = reinterpret_cast<Ctx*>(ctx);
  // the band intermediate doubles as the pass-1 output of the dense transform
  CU(launch_fft_dense(c, reinterpret_cast<const float2*>(d_in), ws_ptr<float2>(c, c->lay.y),
                      reinterpret_cast<float2*>(d_out)));
  return GWMF_OK;
}

int gwmf_uses_fused(const gwmf_ctx* ctx) { return ctx && reinterpret_cast<const Ctx*>(ctx)->fused ? 1 : 0; }

int64_t gwmf_launch_count(const gwmf_ctx* ctx) {
  return ctx ? reinterpret_cast<const Ctx*>(ctx)->launches : 0;
}

const char* gwmf_strerror(int status) {
  switch (status) {
    case GWMF_OK: return "ok";
    case GWMF_E_ARG: return "invalid argument";
    case GWMF_E_EMPTY_TEMPLATE: return "empty template: f_ISCO <= f_low";
    case GWMF_E_STATE: return "bank or segment not loaded";
    case GWMF_E_CAPACITY: return "output buffer too small";
    case GWMF_E_CUDA: return "CUDA error";
    case GWMF_E_WORKSPACE: return "workspace too small";
  }
  return "unknown status";
}

const char* gwmf_last_cuda_error(const gwmf_ctx* ctx) {
  return ctx ? reinterpret_cast<const Ctx*>(ctx)->cuda_err.c_str() : "";
}

}  // extern "C"
