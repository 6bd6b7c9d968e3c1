// gwmf_internal.cuh -- shared declarations of the CUDA side (not part of the C ABI).
#pragma once
#include <cuda.h>           // CUtensorMap (type only; no driver library is linked)
#include <cuda_runtime.h>
#include <stdint.h>
#include <string>
#include <vector>

#include "../../include/gwmf.h"

namespace gwmf {

constexpr int kN2 = 1024;        // second-pass transform length (columns k2), fixed for every N
constexpr int kLogN2 = 10;
constexpr int kMaxBands = 32;
constexpr int kColsPerCta = 8;   // pass-1 column tile: 8 columns x 8 B = 64 B segments per output row
constexpr int kP2Warps = 8;      // pass-2 rows (j1 values) per CTA, one warp each
// Decimated path: a band of at most kSBinsMax bins is transformed on a coarse grid of L <= kLMax points (class S);
// wider bands keep their own n-point transform (class D).  See bandpower.cu.
constexpr int kSBinsMax = 32768; // widest class-S band (bins)
constexpr int kLMax = 16384;     // largest coarse grid one CTA transforms in shared memory
constexpr int kLogLMin = 11;     // smallest coarse grid (2048 points)
constexpr int kSubMax = 4;       // a band that needs L = 2^15 or 2^16 > kLMax points is done as L / kLMax interleaved sub-grids
constexpr int kUCap = kSBinsMax; // entries of the one-sided power spectrum U+ kept per template
// C-major order inside a row of 1024 bins: bin k2 = 32 m + c sits at position 32 c + m (an involution).  The spectra
// the decimated path's first pass reads (Q, U+) are stored this way: its warps read with lane = m.
__host__ __device__ __forceinline__ int cm_pos(int k2) { return ((k2 & 31) << 5) | (k2 >> 5); }

// Per-template record (device).  Phase in TURNS: psi(u) = (((c0 u^2 + c2) u + c3) u + c4) u - 1/8 with
// u = f^(-1/3); this is Psi0/(2 pi) of the 2PN SPA phase (BASELINE.json:configs[0]).
struct TemplateMeta {
  double c0, c2, c3, c4;
  double sigma;                  // Eq. 4, amplitude constant 1
  float scale_rho2;              // (sigma_ref / sigma)^2: rho^2 = |z_scaled|^2 * scale_rho2
  int32_t k_high;                // first bin above the template
  int32_t edges[kMaxBands + 1];  // band l = bins [edges[l], edges[l+1])
  uint32_t wide_mask;            // bit l: band l goes through the generic pass-1 kernel (> 32 input rows)
  uint16_t row_off[kMaxBands + 2];  // band-separated spectrum Qb: rows of narrow band l start at row_off[l] (k_fused)
  // ---- decimated path: the template's EFFECTIVE bands (n-point transforms that are really run) ----
  //   if s_mask != 0:  e = 0: Z = the union of the class-S bands (one transform, gives their share of z)
  //                    e = 1: U = one-sided spectrum of sum_{l in S} |z_l|^2 (real part of its transform), or, for
  //                           the OWNER of a pair (pair == 1), UP = U_A + i U_B, the two-sided spectra of this template
  //                           and of the next one: ONE transform returns u_A + i u_B.  The GUEST (pair == 2) has no
  //                           U band of its own and reads the imaginary part of its owner's.
  //   then one per class-D band in ascending l (z_l itself: contributes to z and to sum |z_l|^2)
  uint32_t s_mask;               // bit l: band l is class S (0 < bins <= s_bins)
  uint32_t d_mask;               // bit l: band l is class D (bins > s_bins)
  uint32_t gen_mask;             // bit e: effective band e has very many input rows and is pre-passed (k_prepass)
  int32_t eff_prefix;            // effective bands of all earlier templates of the bank
  int32_t n_eff;                 // effective bands of this template
  int32_t z_lo, z_hi;            // hull of the class-S bands, bins [z_lo, z_hi)
  int32_t u_hi;                  // support of U+: bins [0, u_hi), u_hi = widest class-S band
  int32_t full_band;             // chi^2 on demand: the ONE effective band is the whole template [edges[0], k_high)
  int32_t pair;                  // 0: unpaired, 1: owner of the pair (t even, t + 1 is its guest), 2: guest
  int32_t up_hi;                 // owner: support of the pair spectrum, bins (-up_hi, up_hi)
};

// One effective band: which spectrum it reads (kind) and the bins [e_lo, e_hi) it owns.
enum EffKind { kEffZ = 0, kEffU = 1, kEffD = 2, kEffUP = 3 };
struct EffBand { int kind, e_lo, e_hi, l; };
// The same, one record per slot of the whole bank (slot = eff_prefix[t] + e), written once per bank setup so that a
// pass-1 CTA finds its work with ONE 32-byte load instead of a search through the template records.
struct alignas(32) SlotDesc {
  int32_t t;                     // template (index into the bank)
  int32_t kind;                  // EffKind
  int32_t e_lo, e_hi;            // bins
  int32_t n_holes;               // Z only: class-D bands inside the hull (0 except for unusual spectra)
  int32_t generic;               // 1: very many input rows: k_prepass reduces them to NA / 32 rounds read from vbuf
  int32_t pad0, pad1;
};
#ifdef __CUDACC__
__device__ __forceinline__ EffBand eff_band(const TemplateMeta* m, int e) {
  EffBand b;
  if (m->full_band) { b.kind = kEffD; b.e_lo = m->edges[0]; b.e_hi = m->k_high; b.l = -1; return b; }
  if (m->s_mask) {
    if (e == 0) { b.kind = kEffZ; b.e_lo = m->z_lo; b.e_hi = m->z_hi; b.l = -1; return b; }
    if (m->pair == 2) {
      e -= 1;                                    // the guest of a pair has no U band of its own
    } else {
      if (e == 1) {
        b.l = -1;
        if (m->pair == 1) { b.kind = kEffUP; b.e_lo = 1 - m->up_hi; b.e_hi = m->up_hi; }
        else { b.kind = kEffU; b.e_lo = 0; b.e_hi = m->u_hi; }
        return b;
      }
      e -= 2;
    }
  }
  unsigned d = m->d_mask;
  for (int i = 0; i < e; ++i) d &= d - 1;
  b.l = __ffs(d) - 1;
  b.kind = kEffD;
  b.e_lo = m->edges[b.l];
  b.e_hi = m->edges[b.l + 1];
  return b;
}
#endif

// One (template, window) trigger slot, updated with a 128-bit compare-and-swap.
//   key  = (bits(rho) << 32) | (0xFFFFFFFF - sample)   -> max key = max rho, lowest sample on ties
//   aux  = bits(chi^2) in the low word
struct alignas(16) Slot {
  unsigned long long key;
  unsigned long long aux;
};

struct Layout {                  // byte offsets into the caller's workspace
  size_t u_tab, c_tab, g_tab, sn, wq, s_in, tw_n1, tw_p2, meta, masks, prefix_totals, slots, counts, offsets, trig_out,
         series_rho, series_chi, flags, q, qb, y, tw_l, wbuf, ubuf, eff, slot_tab, prep, bp_jobs, vbuf, pp_jobs, pw_tab, pw_totals, total;
  size_t y_bytes;
  int batch;                     // most templates per launch
  int y_slots;                   // n-point transforms (n complex fp32 each) the band buffer holds
};

struct Ctx {
  gwmf_params prm;
  int64_t n;
  int log_n;
  int n1;                        // n / kN2
  int na, nb;                    // n1 = na * nb (pass-1 stage radices)
  int k_low;
  int n_windows;
  int n_sms;                     // multiprocessors of the device (persistent-kernel grid size)
  double df;
  Layout lay;
  char* ws;
  cudaStream_t stream;
  cudaStream_t side;             // high-priority side stream for the low-volume pass-1 kernels
  cudaEvent_t ev_fork, ev_join;
  cudaStream_t bp[3];            // decimated path: the band-power kernels of the larger coarse grids run side by side
  cudaEvent_t ev_bp_fork, ev_bp_join[3];
  int n_templates;
  bool have_bank, have_segment;
  int path;                      // GWMF_PATH_TWO_PASS / _FUSED / _DECIMATED (resolved from gwmf_params::path at create)
  bool fused;                    // path == GWMF_PATH_FUSED
  int device;                    // CUDA device the context lives on
  CUtensorMap band_tmap;         // decimated path: the band buffer [tile = slot * NA + ja][c][jb][256 B] as a 4-d tensor (pass 2's row gather)
  int s_bins;                    // decimated path: class-S threshold in bins = min(kSBinsMax, n / 16)
  int t_max;                     // decimated path: effective bands of more than 32 * t_max input rows are pre-passed (k_prepass)
  int32_t* h_eff;                // host mirror (pinned): eff_prefix[0 .. n_templates], then one "has generic band" flag per template
  bool mirror_ready;             // the host mirrors (h_masks, h_eff) have been waited for since the last bank setup
  int64_t launches;
  std::string cuda_err;
  TemplateMeta* h_meta;          // host staging of the bank (pinned)
  std::vector<gwmf_mass_pair> h_masses;   // the loaded bank's masses (gwmf_effective_distance)
  uint32_t* h_masks;             // host mirror of TemplateMeta::wide_mask (pinned), valid once ev_masks has fired
  cudaEvent_t ev_masks;
  // ---- double-buffered segment (s_in, wq): a segment can be uploaded and prepared on the upload stream while the
  // filters of the previous one still run on the main stream (gwmf_load_segment with Sn == NULL)
  int front;                     // buffer the filters read
  bool have_psd;
  bool pending_reset;            // a segment was loaded since the last filter call: the next one clears every slot first
  cudaStream_t upload;
  float* h_stage[2];             // pinned staging of host segments (n floats each)
  cudaEvent_t ev_seg_ready[2];   // wq[b] is complete (recorded on the stream that prepared it)
  cudaEvent_t ev_seg_free[2];    // the last filter launch that reads wq[b] (recorded on the main stream)
  cudaEvent_t ev_stage_free[2];  // the H2D copy out of h_stage[b] is done
  cudaEvent_t ev_last_load;      // end of the latest load (orders the shared preparation scratch between streams)
};
inline float2* wq_buf(Ctx* c, int b) { return reinterpret_cast<float2*>(c->ws + c->lay.wq) + (size_t)b * (size_t)(c->n / 2); }
inline double* pw_buf(Ctx* c, int b) { return reinterpret_cast<double*>(c->ws + c->lay.pw_tab) + (size_t)b * (size_t)(c->n / 2); }   // P[k] of wq[b]
inline float* s_buf(Ctx* c, int b) { return reinterpret_cast<float*>(c->ws + c->lay.s_in) + (size_t)b * (size_t)c->n; }

// ---- launchers (defined in the .cu files) --------------------------------------------------------
cudaError_t launch_tables(Ctx* c);
cudaError_t launch_segment_fft(Ctx* c, int buf, cudaStream_t st);      // s_in[buf] -> data spectrum in the preparation scratch
cudaError_t launch_psd_tables(Ctx* c, cudaStream_t st);                // sn -> g_tab, c_tab, flags
cudaError_t launch_weighted_spectrum(Ctx* c, int buf, cudaStream_t st); // scratch spectrum, sn, c_tab -> wq[buf]
cudaError_t launch_bank_setup(Ctx* c);
cudaError_t launch_pass1_filter(Ctx* c, int first, int count, int next_first, int next_count, int parity, bool q_ready);
cudaError_t launch_correlate(Ctx* c, int first, int count, int parity, cudaStream_t st, bool c_major = false);
cudaError_t launch_correlate_bands(Ctx* c, int first, int count, int parity, cudaStream_t st);
inline int qb_rows_cap(const Ctx* c) { return c->n1 / 2 + kMaxBands + 2; }   // rows of Qb per template
cudaError_t launch_pass1_dense(Ctx* c, const float2* d_in, float2* d_mid, cudaStream_t st);
cudaError_t launch_rowstage_dense(Ctx* c, float2* d_mid, cudaStream_t st);
cudaError_t launch_pass2_filter(Ctx* c, int first, int count, bool update_slots, float* series_rho,
                                float* series_chi);
cudaError_t launch_fused_filter(Ctx* c, int first, int count, int parity, bool update_slots, float* series_rho,
                                float* series_chi);
cudaError_t launch_pass2_dense(Ctx* c, const float2* d_mid, float2* d_out, cudaStream_t st);
inline cudaError_t launch_fft_dense(Ctx* c, const float2* d_in, float2* d_mid, float2* d_out, cudaStream_t st) {
  cudaError_t e = launch_pass1_dense(c, d_in, d_mid, st);
  if (e == cudaSuccess) e = launch_rowstage_dense(c, d_mid, st);
  return e != cudaSuccess ? e : launch_pass2_dense(c, d_mid, d_out, st);
}
// decimated path
cudaError_t configure_pass1(int path);
cudaError_t configure_pass2();
cudaError_t make_band_tensor_map(Ctx* c);   // needs lay.y, n1 (gwmf_create)
cudaError_t configure_bandpower();
size_t bp_jobs_bytes();                      // workspace of the band-power job lists (two batches)
cudaError_t launch_bandpower(Ctx* c, int first, int count, int parity, cudaStream_t st);      // W_l, then U+
cudaError_t launch_pass1_eff(Ctx* c, int first, int count, int parity, cudaStream_t st);
cudaError_t launch_prepass(Ctx* c, int first, int count, int parity, cudaStream_t st);   // bands of very many rows -> vbuf
cudaError_t launch_pass2_eff(Ctx* c, int bfirst, int bcount, int first, int count, bool update_slots, float* series_rho,
                             float* series_chi);
cudaError_t launch_chisq_at_events(Ctx* c, int first, int count, bool loud_only);   // chi^2 from its definition at the events (all, or rho > kRhoLoud)
cudaError_t launch_chisq_series_loud(Ctx* c, int template_id, const float* series_rho, float* series_chi);   // the same for a series
cudaError_t launch_reset_slots(Ctx* c, int first, int count);
cudaError_t launch_compact(Ctx* c);

// The (template, band) pairs of a batch whose bit is set in TemplateMeta::wide_mask, as band indices
// tb * p + l in ascending order, identical in every CTA (so that CTAs can split the list by position).
// s_list: batch * p ints, s_cnt: batch + 1 ints of shared memory.  Returns the list length.
#ifdef __CUDACC__
__device__ inline int build_wide_list(const TemplateMeta* meta, int batch, int p, int* s_list, int* s_cnt) {
  for (int t = threadIdx.x; t < batch; t += blockDim.x) s_cnt[t] = __popc(meta[t].wide_mask);
  __syncthreads();
  if (threadIdx.x == 0) {
    int run = 0;
    for (int t = 0; t < batch; ++t) { const int v = s_cnt[t]; s_cnt[t] = run; run += v; }
    s_cnt[batch] = run;
  }
  __syncthreads();
  for (int t = threadIdx.x; t < batch; t += blockDim.x) {
    unsigned m = meta[t].wide_mask;
    int o = s_cnt[t];
    while (m) { const int l = __ffs(m) - 1; m &= m - 1; s_list[o++] = t * p + l; }
  }
  __syncthreads();
  return s_cnt[batch];
}
#endif
constexpr int kMaxBatch = 128;   // templates per launch (bounds the shared-memory band list)

template <typename T>
inline T* ws_ptr(Ctx* c, size_t off) { return reinterpret_cast<T*>(c->ws + off); }

}  // namespace gwmf
