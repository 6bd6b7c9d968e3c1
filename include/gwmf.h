/* gwmf.h -- C ABI of the B200 inspiral matched-filter + chi^2 hot path (arxiv/paper_0906_4175).
 *
 * What the library computes (citations are PAPER.md lines; readings are listed in DESIGN.md):
 *   z(t)   = 4 int h~_c(f) s~*(f) / S_n(f) e^{2 pi i f t} df                  Eq. 1
 *   rho(t) = |z(t)| / sigma,  sigma^2 = 4 int |h~_c|^2 / S_n df               Eq. 3-4
 *   chi^2(t) = (p/sigma^2) sum_l |z_l(t) - z(t)/p|^2, z_l = Eq. 1 restricted to the l-th of p
 *              frequency bands of equal expected SNR^2                       Eq. 5
 *   templates: 2PN stationary-phase phase, Newtonian f^(-7/6) amplitude, between 40 Hz and
 *              min(f_ISCO, Nyquist)
 *   events: per window of W samples, the sample of maximum rho if rho > threshold, with its
 *           chi^2                                                            PAPER.md:184 (+ DESIGN.md reading 12)
 *
 * Conventions
 *   - Every function returns GWMF_OK (0) or a negative gwmf_status; nothing throws or aborts.
 *   - All device work is enqueued on the CUDA stream given to gwmf_create.  Calls marked "async"
 *     return before the work completes; calls marked "syncs" wait for the stream.
 *   - Ownership: the caller owns every array it passes and the workspace; the library copies what
 *     it needs during the call and owns only the gwmf_ctx.
 *   - One context per stream; calls on one context are not re-entrant.
 *   - There is no CPU fallback: gwmf_create fails with GWMF_E_CUDA if no sm_100 device is current.
 *   - Determinism: identical inputs give bit-identical outputs; triggers come back sorted by
 *     (template_id, window index).
 */
#ifndef GWMF_H
#define GWMF_H

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

/* G Msun / c^3 in seconds (nominal solar mass parameter); masses are in solar masses. */
#define GWMF_T_SUN 4.9254909476412675e-6

typedef enum {
  GWMF_OK = 0,
  GWMF_E_ARG = -1,            /* null pointer, n not a power of two in [2^14, 2^22], p < 1 or > 32,
                                 window not dividing n, non-positive mass, bad S_n                  */
  GWMF_E_EMPTY_TEMPLATE = -2, /* k_high <= k_low: f_ISCO <= f_low (total mass >~ 110 Msun)          */
  GWMF_E_STATE = -3,          /* filter before a bank and a segment are loaded, etc.                */
  GWMF_E_CAPACITY = -4,       /* output buffer too small; *n_out still receives the needed count   */
  GWMF_E_CUDA = -5,           /* a CUDA call failed; gwmf_last_cuda_error() has the text            */
  GWMF_E_WORKSPACE = -6       /* workspace smaller than gwmf_workspace_bytes()                      */
} gwmf_status;

/* Which kernels compute the p band transforms of step a3 (all three compute the same rho, chi^2 and events):
 *   TWO_PASS   pass 1 writes every band's intermediate to HBM (p n complex per template), pass 2 reads it;
 *   FUSED      spill-free: narrow bands are formed inside the row-transform kernel (n <= 2^20);
 *   DECIMATED  bands of at most min(32768, n/16) bins are transformed on a coarse grid of L >= 2 B points, their power
 *              spectra summed, and one n-point transform (shared by two templates) returns sum_l |z_l|^2; only z,
 *              that sum and the wider bands keep n-point transforms (n >= 2^15).  DESIGN.md section 5.
 *   AUTO       the library's choice: DECIMATED for n >= 2^15, TWO_PASS below. */
typedef enum {
  GWMF_PATH_AUTO = 0,
  GWMF_PATH_TWO_PASS = 1,
  GWMF_PATH_FUSED = 2,
  GWMF_PATH_DECIMATED = 3
} gwmf_path;

/* Where chi^2 is evaluated.  EVERY_SAMPLE: chi^2(t) at all n samples (the paper's pipeline; needed
 * for gwmf_series).  ON_DEMAND (the pipeline with the chi^2 loop taken out of the
 * hot path): one full-band transform per template gives rho(t) and the events; chi^2 is then evaluated only at each
 * event's sample, directly from its definition z_l[j] = sum_{k in band l} Q[k] e^{2 pi i jk/n} (one pass over the
 * template's bins per event).  The events carry the same rho, sample and chi^2 up to fp32 rounding.  Decimated path
 * only; gwmf_series then returns rho(t) and leaves chi^2(t) = 0. */
typedef enum {
  GWMF_CHISQ_EVERY_SAMPLE = 0,
  GWMF_CHISQ_ON_DEMAND = 1
} gwmf_chisq_mode;

typedef struct gwmf_ctx gwmf_ctx;                      /* opaque */

typedef struct { double m1, m2; } gwmf_mass_pair;      /* solar masses, > 0, any order */

typedef struct {                                       /* one event, 16 bytes */
  int32_t template_id;                                 /* index into the bank                     */
  int32_t sample;                                      /* j* in [0, n)                            */
  float   rho;                                         /* |z[j*]| / sigma                         */
  float   chisq;                                       /* chi^2[j*], 2p-2 degrees of freedom      */
} gwmf_trigger;

typedef struct {
  int64_t n;             /* samples per segment: power of two, 2^14 .. 2^22 (2^20)   */
  double  fs;            /* sampling rate in Hz (4096)                                            */
  double  f_low;         /* low-frequency cut-off in Hz (40); the bin at exactly f_low is in      */
  int32_t p;             /* chi^2 bands, 1 .. 32 (16)                               */
  double  rho_thresh;    /* SNR threshold, strict '>'                                             */
  int32_t window;        /* W: trigger window in samples, power of two, divides n                 */
  int32_t max_templates; /* capacity of the bank                                                  */
  int32_t batch;         /* most templates filtered per kernel launch, 0 .. 128; sizes the band-intermediate
                            buffer, batch * p * n * 8 bytes, and the correlated spectra, 2 * batch * n * 4 bytes.
                            0 = library default: a band buffer of about 2 GiB; the decimated path then takes up
                            to 128 templates per launch, as many as fit in it (it needs ~2, not p, transforms each).
                            The decimated path processes templates in pairs: an odd value is rounded up            */
  int32_t path;          /* a gwmf_path; GWMF_PATH_AUTO (0) = the library's choice.  A path that does not support n
                            (FUSED: 2^15 .. 2^20, DECIMATED: >= 2^15) is GWMF_E_ARG                               */
  int32_t chisq_mode;    /* a gwmf_chisq_mode; ON_DEMAND needs the decimated path (n >= 2^15), else GWMF_E_ARG     */
} gwmf_params;

/* Bytes of DEVICE memory the caller must provide to gwmf_create (0 if params are invalid). */
size_t gwmf_workspace_bytes(const gwmf_params* params);

/* Create a context.  d_workspace: DEVICE pointer, 256-byte aligned, >= gwmf_workspace_bytes(params),
 * owned by the caller and kept alive until gwmf_destroy.  cuda_stream: a cudaStream_t (NULL = the
 * legacy default stream).  Builds the twiddle tables (async). */
int gwmf_create(const gwmf_params* params, void* d_workspace, size_t workspace_bytes,
                void* cuda_stream, gwmf_ctx** out);

/* Load the template bank: per template the 2PN phase coefficients and
 * k_high = min(ceil(f_cut/df), n/2), f_cut = min(1/(6^1.5 pi M), fs/2).  host_masses: HOST array of
 * n_templates pairs, 1 <= n_templates <= max_templates.  sigma and the p+1 band edges depend on S_n and
 * are (re)computed on the device by gwmf_load_segment / here if a segment is already loaded.  async. */
int gwmf_make_bank(gwmf_ctx* ctx, const gwmf_mass_pair* host_masses, int32_t n_templates);

/* Load one strain segment and, optionally, a new PSD (Eq. 1 inputs).
 *   s  : n fp32 samples of s(t), HOST or DEVICE pointer.
 *   Sn : n/2+1 fp64 samples of the one-sided PSD at f_k = k fs/n, HOST or DEVICE pointer, or NULL = keep the PSD
 *        (and with it sigma and the band edges of every template) of the previous call; the first call must give
 *        one (else GWMF_E_STATE).  Entries below f_low and the Nyquist entry are ignored (Eq. 2 diverges at f -> 0).
 *        Entries inside [f_low, fs/2) must be finite and > 0 -- checked on the device; a violation is reported by
 *        the next syncing call as GWMF_E_ARG.
 * Computes on the device: the data spectrum D[k] = sum_j s[j] e^{-2 pi i jk/n} with the library's own FFT, the
 * weighted spectrum w[k] = (4/n) D[k] f_k^(-7/6) / S_n[k] and, with a new PSD, the fp64 power table
 * C[k] = sum_{k'<=k} f^(-7/3)/S_n (Eq. 4) and sigma and band edges of every loaded template.
 * Ownership: both arrays may be freed as soon as the call returns (host sources are staged before it returns;
 * device sources are read on the context's stream, ordered like any other work the caller puts on that stream).
 * Overlap (the bank sweep of BASELINE.json:configs[3]): the segment buffers are double-buffered.
 * With a HOST segment and Sn == NULL the upload and the transform run on the library's own upload stream, beside
 * filters of the previous segment that are still running; gwmf_filter calls issued AFTER this call use the new
 * segment (they wait for it on the device, not on the host).  The events of the previous segment stay readable by
 * gwmf_triggers until the next gwmf_filter call, so the steady state of a sweep is
 *     gwmf_filter(q);  gwmf_load_segment(q + 1, NULL);  gwmf_triggers(q).
 * With a device segment or a new PSD the work is ordered on the context's stream (no overlap).  async. */
int gwmf_load_segment(gwmf_ctx* ctx, const float* s, const double* Sn);

/* Matched-filter templates [first_template, first_template + n_templates) against the loaded segment
 * (the FIRST call after a bank or PSD change waits on the host for the bank setup to finish: it reads back how
 * many transforms each template needs; later calls do not wait):
 * p band inverse FFTs, rho and chi^2 at every sample (Eq. 3, 5) and the per-window
 * maxima above threshold.  Trigger slots of those templates are reset first.
 * Loud data (reading 23): the transforms' epilogue forms chi^2 in fp32 as sum_l |z_l|^2 - |z|^2 / p, two
 * terms of size rho^2 / p whose difference keeps about rho^2 * 5e-7 of absolute error, and the transforms' own fp32
 * error grows with the mean power of the data in the template's band.  The call therefore re-evaluates chi^2 at the
 * event's sample from Eq. 5 as printed, sum_l |z_l - z/p|^2 with z_l[j] = sum_{k in band l} Q[k] e^{2 pi i jk/n} (one
 * pass over the template's bins per event), for every event with rho > 48 and for every event of a template in whose
 * band the segment's mean power (sum_l |z_l|^2 averaged over the n samples, 2 in noise) exceeds 4 -- a signal of
 * SNR >~ 300 at n = 2^20, matched by that template or not.  gwmf_series applies the same rule per sample.  async. */
int gwmf_filter(gwmf_ctx* ctx, int32_t first_template, int32_t n_templates);

/* Measurement: the same work as gwmf_filter, with CUDA events recorded on the context's stream around the
 * stages of every batch.  host_ms: HOST array of 4 doubles, summed device time (ms) of
 *   [0] the spectra of the decimated path (correlate, coarse-grid band powers, U+), serialised on the main stream
 *       for this call (gwmf_filter runs them beside pass 1 on a side stream); 0 for the other paths, whose
 *       correlate step is inside [1];
 *   [1] pass 1: first FFT pass of every (effective) band -> band intermediate in HBM; for the spill-free path only
 *       the wide bands' kernels;
 *   [2] pass 2: last FFT stage + rho/chi^2/trigger epilogue (spill-free path: k_fused);
 *   [3] chi^2 from its definition at event samples: every event with chisq_mode = ON_DEMAND, otherwise only the
 *       loud ones (see gwmf_filter).
 * host_launches: HOST array of 4 int32, launches / batches timed in each stage.  syncs. */
int gwmf_filter_timed(gwmf_ctx* ctx, int32_t first_template, int32_t n_templates, double* host_ms,
                      int32_t* host_launches);

/* Collect the events of all templates filtered on the segment the last gwmf_filter call used (a gwmf_load_segment
 * issued after that call does not disturb them; the first gwmf_filter on the new segment clears them), sorted by
 * (template_id, window).  host_out: HOST array of `capacity` triggers (may be NULL if capacity = 0).
 * *n_out receives the number of events found; GWMF_E_CAPACITY if it exceeds capacity (nothing is
 * written beyond capacity).  syncs. */
int gwmf_triggers(gwmf_ctx* ctx, gwmf_trigger* host_out, int64_t capacity, int64_t* n_out);

/* sigma of every loaded template (Eq. 4 with unit amplitude constant), HOST array of n_templates
 * doubles.  Needs a bank and a segment.  syncs. */
int gwmf_sigma(gwmf_ctx* ctx, double* host_sigma);

/* Physical amplitude / effective distance (templates carry "Newtonian amplitude" and an "effective
 * distance D_eff from the detector"; the paper prints no constant, reading 4 writes it out):
 *     h~(f) = A f^(-7/6) e^{i Psi(f)},  A(D_eff) = sqrt(5/24) pi^(-2/3) (c / D_eff) (G M_chirp / c^3)^(5/6),
 *     M_chirp = (m1 m2)^(3/5) / (m1 + m2)^(1/5).
 * rho and chi^2 do not depend on A; distances do.  psd_unit is the physical value, in strain^2 / Hz, of ONE unit of
 * the S_n array given to gwmf_load_segment (9e-46 for Eq. 2 as printed; 1 if S_n was already physical).
 * host_d1_mpc: HOST array of n_templates doubles, the effective distance in megaparsecs at which template t has optimal
 * SNR 1 in the loaded PSD: D_1 = A(1 Mpc) sigma / sqrt(psd_unit) (divide by 8 for the usual SNR-8 horizon).
 * Needs a bank and a segment; GWMF_E_ARG for psd_unit <= 0.  syncs. */
int gwmf_effective_distance(gwmf_ctx* ctx, double psd_unit, double* host_d1_mpc);

/* Effective distance of events: host_deff_mpc[i] = D_1[template of event i] / rho_i, the distance at which that template
 * would be seen with the event's SNR.  host_triggers: HOST array of n_triggers events as returned by gwmf_triggers
 * (template_id inside the loaded bank and rho > 0, else GWMF_E_ARG); host_deff_mpc: HOST array of n_triggers doubles.
 * syncs. */
int gwmf_trigger_distances(gwmf_ctx* ctx, double psd_unit, const gwmf_trigger* host_triggers, int64_t n_triggers,
                           double* host_deff_mpc);

/* Band edges e_0..e_p of every loaded template, HOST array of n_templates*(p+1) int32.  syncs. */
int gwmf_band_edges(gwmf_ctx* ctx, int32_t* host_edges);

/* Measurement: the number of n-point transforms the library runs for every loaded template with its path, HOST array
 * of n_templates int32: the non-empty bands (two-pass and spill-free paths), or the effective bands of the
 * decimated path (1 for z + 1 for sum |z_l|^2, which the guest of a template pair does not count, + the number of
 * bands wider than min(32768, n/16) bins; just the bands themselves if fewer than three are narrow).  Each one is n complex fp32 written by pass 1 and read by pass 2: the byte model of bench.py.  syncs. */
int gwmf_transform_counts(gwmf_ctx* ctx, int32_t* host_counts);

/* Debug/parity: full rho(t) and chi^2(t) of one template, n floats each, HOST arrays (either may be
 * NULL).  Runs the same kernels as gwmf_filter on that template with series output enabled; does not
 * touch trigger slots.  syncs. */
int gwmf_series(gwmf_ctx* ctx, int32_t template_id, float* host_rho, float* host_chisq);

/* Debug/parity: the correlate step alone (Eq. 1 integrand).  host_q receives n/2 interleaved
 * complex fp32 values Q[k] = (4/n) D[k] f_k^(-7/6) e^{+i Psi0(f_k)} / (S_n[k] sigma_ref) for k_low <= k < k_high of
 * template `template_id` and 0 elsewhere, with D the forward DFT of the loaded segment and
 * sigma_ref^2 = 4 df sum_{k_low <= k < n/2} f_k^(-7/3)/S_n[k] (the library's internal normalisation, which
 * cancels in rho and chi^2).  HOST array of n floats.  Needs a bank and a segment.  syncs. */
int gwmf_correlate(gwmf_ctx* ctx, int32_t template_id, float* host_q);

/* Debug/parity: the library's batched complex FFT alone.  X[k] = sum_j x[j] e^{+2 pi i jk/n}
 * (unnormalised inverse transform, the e^{2 pi i f t} of Eq. 1).  in/out: DEVICE arrays of n
 * interleaved complex fp32 (re, im), n = params.n; in != out.  async. */
int gwmf_fft_inverse(gwmf_ctx* ctx, const float* d_in, float* d_out);

/* 1 if this context filters with the spill-free kernel (gwmf_params::path = GWMF_PATH_FUSED), else 0. */
int gwmf_uses_fused(const gwmf_ctx* ctx);

/* The gwmf_path this context filters with (GWMF_PATH_AUTO resolved at gwmf_create); GWMF_E_ARG for a null ctx. */
int gwmf_path_in_use(const gwmf_ctx* ctx);

/* The power table of Eq. 4 without a context, a workspace or any allocation:
 *     C[k] = sum_{k' <= k} f_k'^(-7/3) / S_n[k']   over k_low = ceil(f_low n / fs) <= k' <= k,   C[k] = 0 below k_low,
 * from which sigma^2 = 4 (fs/n) C[k_high - 1] and the p + 1 equal-power band edges of any template follow
 * (e_l = 1 + min{k : C[k] >= (l/p) C[k_high - 1]}).  It is the table gwmf_load_segment builds inside its
 * workspace, summed in the same fixed order, so the two agree bit for bit.
 *
 * Meant for callers that must not allocate device memory when the PSD changes: an online search whose running
 * filters a cudaMalloc / cudaFree would stall (both serialise the whole device), a process whose memory a caching
 * allocator or another pipeline already holds, a plug-in that may only touch the buffers it is handed.  The
 * function calls no cudaMalloc, cudaFree or other allocating routine.  Its scratch (1024 partial sums and a status
 * word, GWMF_STATIC_SCRATCH_BYTES in all) is a static array inside the library's device image: every GPU that loads
 * the library carries those bytes until the process exits.
 *
 *   d_sn : DEVICE, n/2 + 1 fp64 samples of the one-sided PSD at f_k = k fs/n (input; entries below f_low and the
 *          Nyquist entry are ignored, the others must be finite and > 0, else GWMF_E_ARG).
 *   d_c  : DEVICE, n/2 fp64 entries (output, fully overwritten; must not overlap d_sn).  Caller-owned, as is d_sn.
 *   n    : power of two, 2^14 .. GWMF_STATIC_MAX_N.  A larger n is refused with GWMF_E_CAPACITY (the scratch and the
 *          kernels' shared-memory tiles are laid out for at most that many samples); other bad values are GWMF_E_ARG.
 *   cuda_stream : a cudaStream_t of the CURRENT device (NULL = legacy default stream); the work runs on it.
 *   err, err_len: optional HOST buffer that receives a one-line description of a failure ("" on success).
 *
 * Runs on the device that is current in the calling thread.  The first call on each device looks up the device
 * address of the static array (cudaGetSymbolAddress; this may also make the driver load the library's device code),
 * so make one call per device at start-up, outside any stream capture; later calls only launch three small kernels.
 * All calls on a device share the one array and it keeps the previous call's contents; the function itself resets the
 * part that must start from zero, on the given stream.  Two calls whose kernels can overlap on the same GPU (different
 * streams, different host threads) race on it: serialise them.  syncs (it reads the status word back). */
#define GWMF_STATIC_MAX_N (1 << 22)
#define GWMF_STATIC_SCRATCH_BYTES 8448
int gwmf_power_table_static(const double* d_sn, double* d_c, int64_t n, double fs, double f_low, void* cuda_stream,
                            char* err, size_t err_len);

/* Number of kernel launches this context has issued so far (for bench.py's gpu_launches). */
int64_t gwmf_launch_count(const gwmf_ctx* ctx);

void gwmf_destroy(gwmf_ctx* ctx);

const char* gwmf_strerror(int status);
const char* gwmf_last_cuda_error(const gwmf_ctx* ctx);   /* "" if none */

#ifdef __cplusplus
}
#endif
#endif /* GWMF_H */
