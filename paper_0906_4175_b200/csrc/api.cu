// api.cu -- the C ABI of include/gwmf.h: argument checking, workspace carving, host-side bank
// arithmetic (phase coefficients, k_high) and the launch sequences.  No compute happens on the host
// beyond a handful of scalars per template.
#include <math.h>
#include <memory>
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
  if (p->path < GWMF_PATH_AUTO || p->path > GWMF_PATH_DECIMATED) return false;
  if (p->path == GWMF_PATH_FUSED && (p->n < (1 << 15) || p->n > (1 << 20))) return false;
  if (p->path == GWMF_PATH_DECIMATED && p->n < (1 << 15)) return false;
  if (p->chisq_mode != GWMF_CHISQ_EVERY_SAMPLE && p->chisq_mode != GWMF_CHISQ_ON_DEMAND) return false;
  if (p->chisq_mode == GWMF_CHISQ_ON_DEMAND && (p->n < (1 << 15) || (p->path != GWMF_PATH_AUTO && p->path != GWMF_PATH_DECIMATED)))
    return false;
  return true;
}

int resolve_path(const gwmf_params* p) {
  // the decimated path needs n1 = n / 1024 >= 32; below that every band goes through the generic two-pass kernels
  if (p->path != GWMF_PATH_AUTO) return p->path;
  return p->n >= (1 << 15) ? GWMF_PATH_DECIMATED : GWMF_PATH_TWO_PASS;
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
  const int path = resolve_path(p);
  L.batch = p->batch > 0 ? p->batch : default_batch(p);
  L.y_slots = L.batch * p->p;
  if (path == GWMF_PATH_DECIMATED && p->batch == 0) {
    // this path needs far fewer than p transforms per template (2 + the wide bands): keep the ~2 GiB band buffer but
    // let a launch take as many templates as fit in it, up to kMaxBatch (launch gaps and kernel tails amortise:
    // measured 116 k -> 124 k template-segments/s from 64 to 128 templates per launch at n = 2^20)
    L.batch = kMaxBatch;
    if (L.y_slots < p->p) L.y_slots = p->p;
  }
  if (L.batch > p->max_templates) L.batch = p->max_templates;
  if (path == GWMF_PATH_DECIMATED && (L.batch & 1)) {
    // templates are processed in pairs (2i, 2i+1 share one transform, segment.cu:k_pairing): a launch holds whole
    // pairs, so an odd limit is rounded up
    L.batch += 1;
    if (L.y_slots < L.batch * p->p && p->batch > 0) L.y_slots = L.batch * p->p;
  }
  size_t off = 0;
  auto take = [&](size_t bytes) { size_t o = off; off = align_up(off + bytes); return o; };
  L.u_tab = take(half * sizeof(double));
  L.c_tab = take(half * sizeof(double));
  L.g_tab = take(half * sizeof(double));
  L.sn = take((half + 1) * sizeof(double));
  L.wq = take(2 * half * sizeof(float2));                      // double-buffered across segments
  L.pw_tab = take(2 * half * sizeof(double));                  // prefix power of each wq buffer (reading 23)
  L.pw_totals = take(2 * 1024 * sizeof(double));
  L.s_in = take(2 * n * sizeof(float));
  L.prep = take(3 * n * sizeof(float2));                       // segment preparation scratch: input, intermediate, transform
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
  L.tw_l = take((size_t)kLMax * sizeof(float2));
  L.eff = take((2 * T + 1) * sizeof(int32_t));
  L.slot_tab = take(path == GWMF_PATH_DECIMATED ? T * (size_t)p->p * sizeof(SlotDesc) : 256);
  L.q = take(2 * (size_t)L.batch * half * sizeof(float2));     // double-buffered across batches
  L.qb = take(path == GWMF_PATH_FUSED ? 2 * (size_t)L.batch * (n1 / 2 + kMaxBands + 2) * kN2 * sizeof(float2) : 256);   // band-separated copy (k_fused)
  // decimated path: per-band one-sided power spectra W_l and their sum U+, double-buffered across batches
  // (not with chi^2 on demand: launch_bandpower never runs there and no effective band reads U+)
  const bool band_powers = path == GWMF_PATH_DECIMATED && p->chisq_mode != GWMF_CHISQ_ON_DEMAND;
  L.wbuf = take(band_powers ? 2 * (size_t)L.batch * (size_t)p->p * kSubMax * kUCap * sizeof(float2) : 256);
  L.ubuf = take(band_powers ? 2 * (size_t)L.batch * kUCap * sizeof(float2) : 256);
  L.bp_jobs = take(band_powers ? bp_jobs_bytes() : 256);
  L.pp_jobs = take((size_t)(L.y_slots + 8) * sizeof(int));
  size_t yb = (size_t)L.y_slots * n * sizeof(float2);
  if (yb < 3 * n * sizeof(float2)) yb = 3 * n * sizeof(float2);   // the dense transform needs in/mid/out
  L.y_bytes = yb;
  L.y = take(yb);
  // pre-passed bands of the decimated path (n1 >= 1024): a twin of the band buffer, slot for slot
  L.vbuf = take(path == GWMF_PATH_DECIMATED && n1 >= 1024 ? (size_t)L.y_slots * n * sizeof(float2) : 256);
  L.total = off;
  return L;
}

bool create_upload_side(Ctx* c) {
  if (cudaStreamCreateWithFlags(&c->upload, cudaStreamNonBlocking) != cudaSuccess) return false;
  if (cudaEventCreateWithFlags(&c->ev_last_load, cudaEventDisableTiming) != cudaSuccess) return false;
  if (cudaEventCreateWithFlags(&c->ev_bp_fork, cudaEventDisableTiming) != cudaSuccess) return false;
  {
    int lo = 0, hi = 0;
    cudaDeviceGetStreamPriorityRange(&lo, &hi);
    for (int i = 0; i < 3; ++i) {
      if (cudaStreamCreateWithPriority(&c->bp[i], cudaStreamNonBlocking, hi) != cudaSuccess) return false;
      if (cudaEventCreateWithFlags(&c->ev_bp_join[i], cudaEventDisableTiming) != cudaSuccess) return false;
    }
  }
  for (int b = 0; b < 2; ++b) {
    if (cudaMallocHost((void**)&c->h_stage[b], sizeof(float) * (size_t)c->n) != cudaSuccess) return false;
    if (cudaEventCreateWithFlags(&c->ev_seg_ready[b], cudaEventDisableTiming) != cudaSuccess) return false;
    if (cudaEventCreateWithFlags(&c->ev_seg_free[b], cudaEventDisableTiming) != cudaSuccess) return false;
    if (cudaEventCreateWithFlags(&c->ev_stage_free[b], cudaEventDisableTiming) != cudaSuccess) return false;
  }
  return true;
}

void destroy_upload_side(Ctx* c) {
  if (c->upload) { cudaStreamSynchronize(c->upload); cudaStreamDestroy(c->upload); c->upload = nullptr; }
  if (c->ev_last_load) cudaEventDestroy(c->ev_last_load);
  if (c->ev_bp_fork) cudaEventDestroy(c->ev_bp_fork);
  for (int i = 0; i < 3; ++i) {
    if (c->bp[i]) { cudaStreamSynchronize(c->bp[i]); cudaStreamDestroy(c->bp[i]); c->bp[i] = nullptr; }
    if (c->ev_bp_join[i]) cudaEventDestroy(c->ev_bp_join[i]);
  }
  for (int b = 0; b < 2; ++b) {
    if (c->h_stage[b]) cudaFreeHost(c->h_stage[b]);
    if (c->ev_seg_ready[b]) cudaEventDestroy(c->ev_seg_ready[b]);
    if (c->ev_seg_free[b]) cudaEventDestroy(c->ev_seg_free[b]);
    if (c->ev_stage_free[b]) cudaEventDestroy(c->ev_stage_free[b]);
  }
}

int fail_cuda(Ctx* c, cudaError_t e, int line = 0) {
  c->cuda_err = cudaGetErrorString(e);
  if (line) c->cuda_err += " (api.cu:" + std::to_string(line) + ")";
  return GWMF_E_CUDA;
}

#define CU(call)                                                 \
  do {                                                           \
    cudaError_t e__ = (call);                                    \
    if (e__ != cudaSuccess) return fail_cuda(c, e__, __LINE__);  \
  } while (0)

// Every entry point runs on the context's device whatever device is current in the calling thread, and restores
// the caller's device on return.
struct DeviceGuard {
  int prev = -1;
  bool switched = false;
  explicit DeviceGuard(int dev) {
    if (cudaGetDevice(&prev) == cudaSuccess && prev != dev) switched = cudaSetDevice(dev) == cudaSuccess;
  }
  ~DeviceGuard() { if (switched) cudaSetDevice(prev); }
};

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
  c->path = resolve_path(params);
  c->fused = c->path == GWMF_PATH_FUSED;
  c->device = dev;
  c->s_bins = (int)(params->n / 16 < kSBinsMax ? params->n / 16 : kSBinsMax);
  // rounds of 32 input rows beyond which k_prepass pays (it leaves Q = NA / 32 rounds and costs about one transform's traffic)
  c->t_max = c->n1 >= 1024 ? c->n1 / 1024 + 5 : (1 << 20);
  c->launches = 0;
  c->h_meta = nullptr;
  c->h_masks = nullptr;
  c->h_eff = nullptr;
  c->mirror_ready = false;
  c->front = 0;
  c->have_psd = false;
  c->pending_reset = false;
  c->upload = nullptr;
  c->ev_last_load = nullptr;
  c->ev_bp_fork = nullptr;
  for (int i = 0; i < 3; ++i) { c->bp[i] = nullptr; c->ev_bp_join[i] = nullptr; }
  for (int b = 0; b < 2; ++b) { c->h_stage[b] = nullptr; c->ev_seg_ready[b] = c->ev_seg_free[b] = c->ev_stage_free[b] = nullptr; }
  // > 48 KB of dynamic shared memory is an opt-in per function AND per device: do it for this context's device
  if (configure_pass1(c->path) != cudaSuccess || configure_pass2() != cudaSuccess || configure_bandpower() != cudaSuccess ||
      (c->path == GWMF_PATH_DECIMATED && make_band_tensor_map(c) != cudaSuccess)) {
    delete c;
    return GWMF_E_CUDA;
  }
  c->side = nullptr;
  c->ev_fork = c->ev_join = c->ev_masks = nullptr;
  {
    int lo = 0, hi = 0;
    cudaDeviceGetStreamPriorityRange(&lo, &hi);
    if (cudaStreamCreateWithPriority(&c->side, cudaStreamNonBlocking, hi) != cudaSuccess ||
        cudaEventCreateWithFlags(&c->ev_fork, cudaEventDisableTiming) != cudaSuccess ||
        cudaEventCreateWithFlags(&c->ev_join, cudaEventDisableTiming) != cudaSuccess ||
        cudaEventCreateWithFlags(&c->ev_masks, cudaEventDisableTiming) != cudaSuccess ||
        cudaMallocHost((void**)&c->h_masks, sizeof(uint32_t) * (size_t)params->max_templates) != cudaSuccess ||
        cudaMallocHost((void**)&c->h_eff, sizeof(int32_t) * (size_t)(2 * params->max_templates + 1)) != cudaSuccess ||
        !create_upload_side(c)) {
      destroy_upload_side(c);
      if (c->side) cudaStreamDestroy(c->side);
      if (c->ev_fork) cudaEventDestroy(c->ev_fork);
      if (c->ev_join) cudaEventDestroy(c->ev_join);
      if (c->ev_masks) cudaEventDestroy(c->ev_masks);
      if (c->h_masks) cudaFreeHost(c->h_masks);
      if (c->h_eff) cudaFreeHost(c->h_eff);
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
  DeviceGuard guard(c->device);
  cudaStreamSynchronize(c->stream);
  destroy_upload_side(c);
  if (c->side) { cudaStreamSynchronize(c->side); cudaStreamDestroy(c->side); }
  if (c->ev_fork) cudaEventDestroy(c->ev_fork);
  if (c->ev_join) cudaEventDestroy(c->ev_join);
  if (c->ev_masks) cudaEventDestroy(c->ev_masks);
  if (c->h_masks) cudaFreeHost(c->h_masks);
  if (c->h_eff) cudaFreeHost(c->h_eff);
  if (c->h_meta) cudaFreeHost(c->h_meta);
  delete c;
}

int gwmf_make_bank(gwmf_ctx* ctx, const gwmf_mass_pair* host_masses, int32_t n_templates) {
  if (!ctx || !host_masses) return GWMF_E_ARG;
  Ctx* c = reinterpret_cast<Ctx*>(ctx);
  DeviceGuard guard(c->device);
  if (n_templates < 1 || n_templates > c->prm.max_templates) return GWMF_E_ARG;
  // Failure-atomic: h_meta is also the host mirror launch_correlate trims its grid with (k_high), so a bank that is
  // rejected half way must leave it -- like the device bank, n_templates and have_bank -- describing the old bank.
  std::unique_ptr<TemplateMeta[]> fresh(new (std::nothrow) TemplateMeta[(size_t)n_templates]);
  if (!fresh) return GWMF_E_ARG;
  for (int t = 0; t < n_templates; ++t) {
    int rc = fill_template(c, host_masses[t], &fresh[(size_t)t]);
    if (rc != GWMF_OK) return rc;
  }
  CU(cudaStreamSynchronize(c->stream));            // h_meta may still be in flight from a previous call
  memcpy(c->h_meta, fresh.get(), sizeof(TemplateMeta) * (size_t)n_templates);
  try { c->h_masses.assign(host_masses, host_masses + n_templates); } catch (...) { return GWMF_E_ARG; }
  CU(cudaMemcpyAsync(ws_ptr<TemplateMeta>(c, c->lay.meta), c->h_meta, sizeof(TemplateMeta) * (size_t)n_templates,
                     cudaMemcpyHostToDevice, c->stream));
  c->n_templates = n_templates;
  c->have_bank = true;
  CU(launch_reset_slots(c, 0, c->prm.max_templates));
  if (c->have_segment) {
    CU(cudaStreamWaitEvent(c->stream, c->ev_last_load, 0));   // the PSD tables of a load that ran on the upload stream
    CU(launch_bank_setup(c));
  }
  return GWMF_OK;
}

int gwmf_load_segment(gwmf_ctx* ctx, const float* s, const double* Sn) {
  if (!ctx || !s) return GWMF_E_ARG;
  Ctx* c = reinterpret_cast<Ctx*>(ctx);
  DeviceGuard guard(c->device);
  if (!Sn && !c->have_psd) return GWMF_E_STATE;               // "same PSD" needs an earlier call that gave one
  cudaPointerAttributes at;
  const bool dev_s = cudaPointerGetAttributes(&at, s) == cudaSuccess && at.type == cudaMemoryTypeDevice;
  cudaGetLastError();
  const int back = c->have_segment ? c->front ^ 1 : 0;
  const size_t s_bytes = sizeof(float) * (size_t)c->n;
  // A host segment with an unchanged PSD is uploaded and transformed on the upload stream, beside the filters of the
  // previous segment.  Everything else (device sources; a new PSD, which rewrites tables the filters read) is simply
  // ordered on the main stream.
  const bool overlapped = !dev_s && !Sn;
  cudaStream_t st = overlapped ? c->upload : c->stream;
  if (overlapped) {
    CU(cudaEventSynchronize(c->ev_stage_free[back]));           // the staging buffer's previous upload (long done)
    memcpy(c->h_stage[back], s, s_bytes);                       // the caller's array is free again on return
    CU(cudaStreamWaitEvent(st, c->ev_seg_free[back], 0));       // filters that still read s_in / wq[back]
    CU(cudaStreamWaitEvent(st, c->ev_last_load, 0));            // the preparation scratch
    CU(cudaMemcpyAsync(s_buf(c, back), c->h_stage[back], s_bytes, cudaMemcpyHostToDevice, st));
    CU(cudaEventRecord(c->ev_stage_free[back], st));
  } else {
    CU(cudaStreamWaitEvent(st, c->ev_last_load, 0));
    CU(cudaMemcpyAsync(s_buf(c, back), s, s_bytes, cudaMemcpyDefault, st));
    if (Sn)
      CU(cudaMemcpyAsync(ws_ptr<double>(c, c->lay.sn), Sn, sizeof(double) * (size_t)(c->n / 2 + 1), cudaMemcpyDefault, st));
    // pinned host sources are copied truly asynchronously: wait so that the caller may free them on return
    bool dev_p = true;
    if (Sn) { dev_p = cudaPointerGetAttributes(&at, Sn) == cudaSuccess && at.type == cudaMemoryTypeDevice; cudaGetLastError(); }
    if (!dev_s || !dev_p) CU(cudaStreamSynchronize(st));
  }
  CU(launch_segment_fft(c, back, st));
  if (Sn) CU(launch_psd_tables(c, st));
  CU(launch_weighted_spectrum(c, back, st));
  CU(cudaEventRecord(c->ev_seg_ready[back], st));
  CU(cudaEventRecord(c->ev_last_load, st));
  c->front = back;
  c->have_segment = true;
  c->pending_reset = true;                                     // events of the previous segment stay readable until the next filter
  if (Sn) {
    c->have_psd = true;
    if (c->have_bank) CU(launch_bank_setup(c));
  }
  return GWMF_OK;
}

// Before any work that reads the current segment's weighted spectrum on the main stream.
static int begin_segment_use(Ctx* c) {
  CU(cudaStreamWaitEvent(c->stream, c->ev_seg_ready[c->front], 0));
  return GWMF_OK;
}
static int end_segment_use(Ctx* c) {
  CU(cudaEventRecord(c->ev_seg_free[c->front], c->stream));
  return GWMF_OK;
}

// ---- host mirrors of the per-template masks / effective-band counts (written by the bank setup) ----
// Waited for ONCE after every bank setup, not per call.
static int ensure_mirror(Ctx* c) {
  if (!c->mirror_ready) {
    CU(cudaEventSynchronize(c->ev_masks));
    c->mirror_ready = true;
  }
  return GWMF_OK;
}

// Q, W_l and U+ of a batch (decimated path), on stream st
static cudaError_t launch_spectra(Ctx* c, int first, int count, int parity, cudaStream_t st) {
  cudaError_t e = launch_correlate(c, first, count, parity, st, true);
  if (e == cudaSuccess && c->prm.chisq_mode != GWMF_CHISQ_ON_DEMAND) e = launch_bandpower(c, first, count, parity, st);
  return e;
}

static bool any_generic(const Ctx* c, int first, int count) {
  for (int t = first; t < first + count; ++t)
    if (c->h_eff[c->n_templates + 1 + t]) return true;
  return false;
}

// One batch of the decimated path: [bfirst, bfirst + bcount) is pair-aligned (whole pairs 2i, 2i+1: spectra and pass 1
// run for all of it), pass 2 processes the rows of [first, first + count) inside it.  Main stream: pass 1 of the
// effective bands, pass 2.  Side stream (high priority, between a fork and a join): the generic kernel for the very
// wide bands of THIS batch, then the spectra (correlate, band powers) of the NEXT batch into the other half of the
// double buffers.
//   ev: optional 4 events (timed mode: everything serialised on the main stream) recorded before the spectra,
//   before pass 1, before pass 2 and after pass 2.
struct Batch { int bfirst, bcount, first, count; };

static cudaError_t decimated_batch(Ctx* c, const Batch& b, const Batch* nx, int parity, bool ready, bool update_slots,
                                   float* series_rho, float* series_chi, cudaEvent_t* ev) {
  cudaError_t e;
  const bool gen = any_generic(c, b.bfirst, b.bcount);
  if (ev) {
    if ((e = cudaEventRecord(ev[0], c->stream)) != cudaSuccess) return e;
    if ((e = launch_spectra(c, b.bfirst, b.bcount, parity, c->stream)) != cudaSuccess) return e;
    if ((e = cudaEventRecord(ev[1], c->stream)) != cudaSuccess) return e;
    if (gen && (e = launch_prepass(c, b.bfirst, b.bcount, parity, c->stream)) != cudaSuccess) return e;
    if ((e = launch_pass1_eff(c, b.bfirst, b.bcount, parity, c->stream)) != cudaSuccess) return e;
    if ((e = cudaEventRecord(ev[2], c->stream)) != cudaSuccess) return e;
    if ((e = launch_pass2_eff(c, b.bfirst, b.bcount, b.first, b.count, update_slots, series_rho, series_chi)) != cudaSuccess) return e;
    return cudaEventRecord(ev[3], c->stream);
  }
  if (!ready && (e = launch_spectra(c, b.bfirst, b.bcount, parity, c->stream)) != cudaSuccess) return e;
  const bool side_work = nx != nullptr;
  if (side_work) {
    // fork: everything enqueued so far on the main stream (this batch's spectra, the previous batch's pass 2, which
    // read the band buffer and the other half of the spectra buffers) precedes the side work
    if ((e = cudaEventRecord(c->ev_fork, c->stream)) != cudaSuccess) return e;
    if ((e = cudaStreamWaitEvent(c->side, c->ev_fork, 0)) != cudaSuccess) return e;
    if (nx && (e = launch_spectra(c, nx->bfirst, nx->bcount, parity ^ 1, c->side)) != cudaSuccess) return e;
    if ((e = cudaEventRecord(c->ev_join, c->side)) != cudaSuccess) return e;
  }
  if (gen && (e = launch_prepass(c, b.bfirst, b.bcount, parity, c->stream)) != cudaSuccess) return e;
  if ((e = launch_pass1_eff(c, b.bfirst, b.bcount, parity, c->stream)) != cudaSuccess) return e;
  if ((e = launch_pass2_eff(c, b.bfirst, b.bcount, b.first, b.count, update_slots, series_rho, series_chi)) != cudaSuccess) return e;
  // join: the next batch's spectra may run beside BOTH passes of this batch (they fill the kernels' tails); the main
  // stream only needs them before the next batch's first pass
  if (side_work && (e = cudaStreamWaitEvent(c->stream, c->ev_join, 0)) != cudaSuccess) return e;
  return cudaSuccess;
}

// Cut [first, first + n) into launches: at most lay.batch templates each and, on the decimated path, at most
// lay.y_slots n-point transforms (the band buffer's capacity) over whole pairs of templates; needs the host mirror.
static void partition(const Ctx* c, int first, int n, std::vector<Batch>& out) {
  out.clear();
  const int end = first + n;
  if (c->path != GWMF_PATH_DECIMATED) {
    for (int t = first; t < end; t += c->lay.batch) {
      const int cnt = end - t < c->lay.batch ? end - t : c->lay.batch;
      out.push_back(Batch{t, cnt, t, cnt});
    }
    return;
  }
  const int T = c->n_templates;
  int t = first & ~1;                                 // pair-aligned start
  while (t < end) {
    int cnt = 0;
    while (t + cnt < end && cnt + 2 <= c->lay.batch) {
      const int step = t + cnt + 2 <= T ? 2 : 1;      // the last template of an odd bank stands alone
      if (c->h_eff[t + cnt + step] - c->h_eff[t] > c->lay.y_slots) break;
      cnt += step;
    }
    if (cnt == 0) cnt = t + 2 <= T ? 2 : 1;           // cannot happen: a pair needs at most 2 p <= y_slots
    const int lo = t > first ? t : first, hi = t + cnt < end ? t + cnt : end;
    out.push_back(Batch{t, cnt, lo, hi - lo});
    t += cnt;
  }
}

// All batches of [first_template, first_template + n_templates).  ev: 4 events per batch (timed mode) or nullptr.
static int run_batches(Ctx* c, int first_template, int n_templates, cudaEvent_t* ev, const std::vector<Batch>& batches) {
  int rc = begin_segment_use(c);
  if (rc != GWMF_OK) return rc;
  if (c->pending_reset) {                       // first filter call on a new segment: forget the previous segment's events
    CU(launch_reset_slots(c, 0, c->prm.max_templates));
    c->pending_reset = false;
  }
  CU(launch_reset_slots(c, first_template, n_templates));
  int parity = 0;
  for (size_t b = 0; b < batches.size(); ++b, parity ^= 1) {
    const Batch& bt = batches[b];
    const Batch* nx = b + 1 < batches.size() ? &batches[b + 1] : nullptr;
    cudaEvent_t* evb = ev ? ev + 4 * b : nullptr;
    if (c->path == GWMF_PATH_DECIMATED) {
      CU(decimated_batch(c, bt, nx, parity, b > 0, true, nullptr, nullptr, evb));
    } else {
      if (evb) CU(cudaEventRecord(evb[0], c->stream));
      if (evb) CU(cudaEventRecord(evb[1], c->stream));
      CU(launch_pass1_filter(c, bt.first, bt.count, nx ? nx->first : 0, nx ? nx->count : 0, parity, b > 0));
      if (evb) CU(cudaEventRecord(evb[2], c->stream));
      if (c->fused) CU(launch_fused_filter(c, bt.first, bt.count, parity, true, nullptr, nullptr));
      else CU(launch_pass2_filter(c, bt.first, bt.count, true, nullptr, nullptr));
      if (evb) CU(cudaEventRecord(evb[3], c->stream));
    }
  }
  // chi^2 from its definition (Eq. 5 as printed): at every event with chi^2 on demand, else at the loud ones, where the
  // epilogue's fp32 difference sum |z_l|^2 - |z|^2 / p has lost its digits (readings 21, 23)
  {
    const bool on_demand = c->prm.chisq_mode == GWMF_CHISQ_ON_DEMAND;
    if (ev) CU(cudaEventRecord(ev[4 * batches.size()], c->stream));
    CU(launch_chisq_at_events(c, first_template, n_templates, !on_demand));
    if (ev) CU(cudaEventRecord(ev[4 * batches.size() + 1], c->stream));
  }
  return end_segment_use(c);
}

static bool range_ok(const Ctx* c, int32_t first_template, int32_t n_templates) {
  return first_template >= 0 && n_templates >= 0 && first_template <= c->n_templates &&
         n_templates <= c->n_templates - first_template;          // no signed overflow for hostile arguments
}

int gwmf_filter(gwmf_ctx* ctx, int32_t first_template, int32_t n_templates) {
  if (!ctx) return GWMF_E_ARG;
  Ctx* c = reinterpret_cast<Ctx*>(ctx);
  DeviceGuard guard(c->device);
  if (!c->have_bank || !c->have_segment) return GWMF_E_STATE;
  if (!range_ok(c, first_template, n_templates)) return GWMF_E_ARG;
  if (n_templates == 0) return GWMF_OK;
  int rc = ensure_mirror(c);
  if (rc != GWMF_OK) return rc;
  std::vector<Batch> batches;
  partition(c, first_template, n_templates, batches);
  return run_batches(c, first_template, n_templates, nullptr, batches);
}

int gwmf_filter_timed(gwmf_ctx* ctx, int32_t first_template, int32_t n_templates, double* host_ms,
                      int32_t* host_launches) {
  if (!ctx || !host_ms || !host_launches) return GWMF_E_ARG;
  Ctx* c = reinterpret_cast<Ctx*>(ctx);
  DeviceGuard guard(c->device);
  if (!c->have_bank || !c->have_segment) return GWMF_E_STATE;
  if (!range_ok(c, first_template, n_templates) || n_templates < 1) return GWMF_E_ARG;
  int rc = ensure_mirror(c);
  if (rc != GWMF_OK) return rc;
  std::vector<Batch> batches;
  partition(c, first_template, n_templates, batches);
  const int nb = (int)batches.size();
  struct Events {                                   // destroyed on every exit path
    std::vector<cudaEvent_t> v;
    ~Events() { for (cudaEvent_t e : v) if (e) cudaEventDestroy(e); }
  } ev;
  ev.v.assign((size_t)nb * 4 + 2, nullptr);
  for (auto& e : ev.v) CU(cudaEventCreate(&e));
  rc = run_batches(c, first_template, n_templates, ev.v.data(), batches);
  if (rc != GWMF_OK) return rc;
  CU(cudaStreamSynchronize(c->stream));
  host_ms[0] = host_ms[1] = host_ms[2] = 0.0;
  for (int b = 0; b < nb; ++b)
    for (int i = 0; i < 3; ++i) {
      float m = 0.f;
      CU(cudaEventElapsedTime(&m, ev.v[4 * b + i], ev.v[4 * b + i + 1]));
      host_ms[i] += m;
    }
  host_launches[0] = c->path == GWMF_PATH_DECIMATED ? nb : 0;
  host_launches[1] = host_launches[2] = nb;
  {
    float m = 0.f;
    CU(cudaEventElapsedTime(&m, ev.v[4 * nb], ev.v[4 * nb + 1]));
    host_ms[3] = m;
    host_launches[3] = c->prm.chisq_mode == GWMF_CHISQ_ON_DEMAND ? (n_templates + 65534) / 65535 : 1;
  }
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
  DeviceGuard guard(c->device);
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
  DeviceGuard guard(c->device);
  std::vector<TemplateMeta> v;
  int rc = fetch_meta(c, v);
  if (rc != GWMF_OK) return rc;
  for (size_t t = 0; t < v.size(); ++t) host_sigma[t] = v[t].sigma;
  return GWMF_OK;
}

// Physical amplitude of template (m1, m2) at 1 Mpc ("Newtonian amplitude", "effective distance"; the constant
// is SURVEY.md 8(c2) reading 4): sqrt(5/24) pi^(-2/3) (c / 1 Mpc) (T_sun M_chirp)^(5/6), host scalars like fill_template.
static double amplitude_1mpc(const gwmf_mass_pair& mp) {
  const double pi = 3.14159265358979323846;
  const double c_over_mpc = 299792458.0 / 3.0856775814913673e22;              // 1/s
  const double mt = mp.m1 + mp.m2, eta = mp.m1 * mp.m2 / (mt * mt);
  const double mchirp_s = GWMF_T_SUN * mt * pow(eta, 0.6);                    // chirp mass in seconds
  return sqrt(5.0 / 24.0) / cbrt(pi * pi) * c_over_mpc * pow(mchirp_s, 5.0 / 6.0);
}

int gwmf_effective_distance(gwmf_ctx* ctx, double psd_unit, double* host_d1_mpc) {
  if (!ctx || !host_d1_mpc || !(psd_unit > 0.0) || !isfinite(psd_unit)) return GWMF_E_ARG;
  Ctx* c = reinterpret_cast<Ctx*>(ctx);
  DeviceGuard guard(c->device);
  std::vector<TemplateMeta> v;
  int rc = fetch_meta(c, v);
  if (rc != GWMF_OK) return rc;
  const double inv_root = 1.0 / sqrt(psd_unit);
  for (size_t t = 0; t < v.size(); ++t) host_d1_mpc[t] = amplitude_1mpc(c->h_masses[t]) * v[t].sigma * inv_root;
  return GWMF_OK;
}

int gwmf_trigger_distances(gwmf_ctx* ctx, double psd_unit, const gwmf_trigger* host_triggers, int64_t n_triggers,
                           double* host_deff_mpc) {
  if (!ctx || n_triggers < 0 || (n_triggers > 0 && (!host_triggers || !host_deff_mpc))) return GWMF_E_ARG;
  if (!(psd_unit > 0.0) || !isfinite(psd_unit)) return GWMF_E_ARG;
  Ctx* c = reinterpret_cast<Ctx*>(ctx);
  DeviceGuard guard(c->device);
  for (int64_t i = 0; i < n_triggers; ++i)
    if (host_triggers[i].template_id < 0 || host_triggers[i].template_id >= c->n_templates || !(host_triggers[i].rho > 0.f))
      return GWMF_E_ARG;
  std::vector<TemplateMeta> v;
  int rc = fetch_meta(c, v);
  if (rc != GWMF_OK) return rc;
  const double inv_root = 1.0 / sqrt(psd_unit);
  for (int64_t i = 0; i < n_triggers; ++i) {
    const int t = host_triggers[i].template_id;
    host_deff_mpc[i] = amplitude_1mpc(c->h_masses[(size_t)t]) * v[(size_t)t].sigma * inv_root / (double)host_triggers[i].rho;
  }
  return GWMF_OK;
}

int gwmf_transform_counts(gwmf_ctx* ctx, int32_t* host_counts) {
  if (!ctx || !host_counts) return GWMF_E_ARG;
  Ctx* c = reinterpret_cast<Ctx*>(ctx);
  DeviceGuard guard(c->device);
  std::vector<TemplateMeta> v;
  int rc = fetch_meta(c, v);
  if (rc != GWMF_OK) return rc;
  const int p = c->prm.p;
  for (size_t t = 0; t < v.size(); ++t) {
    if (c->path == GWMF_PATH_DECIMATED) { host_counts[t] = v[t].n_eff; continue; }
    int cnt = 0;
    for (int l = 0; l < p; ++l) cnt += v[t].edges[l + 1] > v[t].edges[l] ? 1 : 0;
    host_counts[t] = cnt;
  }
  return GWMF_OK;
}

int gwmf_band_edges(gwmf_ctx* ctx, int32_t* host_edges) {
  if (!ctx || !host_edges) return GWMF_E_ARG;
  Ctx* c = reinterpret_cast<Ctx*>(ctx);
  DeviceGuard guard(c->device);
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
  DeviceGuard guard(c->device);
  if (!c->have_bank || !c->have_segment) return GWMF_E_STATE;
  if (template_id < 0 || template_id >= c->n_templates) return GWMF_E_ARG;
  int rc = check_flags(c);
  if (rc != GWMF_OK) return rc;
  float* d_rho = ws_ptr<float>(c, c->lay.series_rho);
  float* d_chi = ws_ptr<float>(c, c->lay.series_chi);
  rc = ensure_mirror(c);
  if (rc != GWMF_OK) return rc;
  if ((rc = begin_segment_use(c)) != GWMF_OK) return rc;
  if (c->path == GWMF_PATH_DECIMATED) {
    const bool on_demand = c->prm.chisq_mode == GWMF_CHISQ_ON_DEMAND;          // no chi^2(t) series in that mode
    if (on_demand) CU(cudaMemsetAsync(d_chi, 0, sizeof(float) * (size_t)c->n, c->stream));
    std::vector<Batch> one;
    partition(c, template_id, 1, one);                                         // the template's pair, rows of the template
    CU(decimated_batch(c, one[0], nullptr, 0, false, false, d_rho, on_demand ? nullptr : d_chi, nullptr));
  } else {
    CU(launch_pass1_filter(c, template_id, 1, 0, 0, 0, false));
    if (c->fused) CU(launch_fused_filter(c, template_id, 1, 0, false, d_rho, d_chi));
    else CU(launch_pass2_filter(c, template_id, 1, false, d_rho, d_chi));
  }
  if (c->prm.chisq_mode != GWMF_CHISQ_ON_DEMAND) CU(launch_chisq_series_loud(c, template_id, d_rho, d_chi));
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
  DeviceGuard guard(c->device);
  if (!c->have_bank || !c->have_segment) return GWMF_E_STATE;
  if (template_id < 0 || template_id >= c->n_templates) return GWMF_E_ARG;
  int rc = check_flags(c);
  if (rc != GWMF_OK) return rc;
  const size_t half = (size_t)(c->n / 2);
  float2* d_q = ws_ptr<float2>(c, c->lay.q);
  if ((rc = begin_segment_use(c)) != GWMF_OK) return rc;
  CU(cudaMemsetAsync(d_q, 0, half * sizeof(float2), c->stream));      // bins outside [k_low, k_high) are not written
  CU(launch_correlate(c, template_id, 1, 0, c->stream));
  CU(cudaMemcpyAsync(host_q, d_q, half * sizeof(float2), cudaMemcpyDeviceToHost, c->stream));
  CU(cudaStreamSynchronize(c->stream));
  return GWMF_OK;
}

int gwmf_fft_inverse(gwmf_ctx* ctx, const float* d_in, float* d_out) {
  if (!ctx || !d_in || !d_out || d_in == d_out) return GWMF_E_ARG;
  Ctx* c = reinterpret_cast<Ctx*>(ctx);
  DeviceGuard guard(c->device);
  // the band intermediate doubles as the pass-1 output of the dense transform
  CU(launch_fft_dense(c, reinterpret_cast<const float2*>(d_in), ws_ptr<float2>(c, c->lay.y),
                      reinterpret_cast<float2*>(d_out), c->stream));
  return GWMF_OK;
}

int gwmf_uses_fused(const gwmf_ctx* ctx) { return ctx && reinterpret_cast<const Ctx*>(ctx)->fused ? 1 : 0; }

int gwmf_path_in_use(const gwmf_ctx* ctx) { return ctx ? reinterpret_cast<const Ctx*>(ctx)->path : GWMF_E_ARG; }

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
