// pass2.cu -- last 32-point stage of the band inverse FFTs fused with the statistics and the trigger
// maxima (end of step a3, steps a4 and a5).
//
// Index algebra (see pass1.cu): sample j = j1 + n1 (jm + 32 jc); pass 1 leaves, per band l and row j1,
//     A_l[j1][c][jm] = sum_m e^{2 pi i jm m/32} Y_l[j1][32 m + c]                              (8 KB, contiguous)
// so that        z_l[j1 + n1 (jm + 32 jc)] = sum_c e^{2 pi i jc c/32} e^{2 pi i jm c/1024} A_l[j1][c][jm]
// is ONE twiddle multiply (table in shared memory, same for every row and band) and ONE 32-point
// transform per thread with lane = jm: no transpose, no shared-memory exchange.  Warps are persistent: a warp walks over rows (template, j1) and, within a row, over the p
// bands; every 8 KB row is brought into the warp's ring of shared-memory buffers by one TMA bulk copy
// (cp.async.bulk + mbarrier), issued kP2Ring rows ahead across band AND row boundaries, so HBM latency is
// hidden by the ring, not by occupancy.  Per owned output sample the warp accumulates
//     z   = sum_l z_l            (Sigma_l z_l = z: no separate full-band transform)
//     q   = sum_l |z_l|^2
// so that rho^2 = |z|^2 / sigma^2 (Eq. 3) and chi^2 = (p/sigma^2)(q - |z|^2/p), which is Eq. 5
// by the identity sum_l |z_l - z/p|^2 = sum_l |z_l|^2 - |z|^2/p.  The band series never
// reach HBM.  Samples with rho > threshold race for their (template, window) slot with a 128-bit
// compare-and-swap on (rho, -index | chi^2): the result is the maximum, lowest index on ties,
// whatever the order of arrival.
#include <string.h>

#include <cuda.h>          // CUtensorMap (types only: the encoder is fetched through cudaGetDriverEntryPoint)

#include "fft_reg.cuh"
#include "gwmf_internal.cuh"

namespace gwmf {

struct P2Args {
  const float2* y;            // A layout: [batch][p][n1][c = 32][jm = 32]
  const float2* tw_p2;        // [32][32] e^{2 pi i c jm/1024}
  const TemplateMeta* meta;   // offset to first template of the batch
  Slot* slots;                // offset to first template of the batch; nullptr = do not update
  float* series_rho;          // optional: n floats (batch must be 1)
  float* series_chi;
  float2* dense_out;          // STORE mode: n complex
  int p;
  int n1;
  int log_n1;
  int log_w;                  // log2(window)
  int n_windows;
  int n_rows;                 // rows (template, j1) of this launch = batch * n1
  float thresh;
};

__device__ __forceinline__ void slot_max(Slot* s, unsigned long long key, unsigned long long aux) {
  unsigned long long old_k = 0ull, old_a = 0ull;    // optimistic guess: the slot is still empty
  while (true) {
    unsigned long long got_k, got_a;
    asm volatile(
        "{\n\t"
        ".reg .b128 cmp, swp, old;\n\t"
        "mov.b128 cmp, {%2, %3};\n\t"
        "mov.b128 swp, {%4, %5};\n\t"
        "atom.global.relaxed.gpu.cas.b128 old, [%6], cmp, swp;\n\t"
        "mov.b128 {%0, %1}, old;\n\t"
        "}"
        : "=l"(got_k), "=l"(got_a)
        : "l"(old_k), "l"(old_a), "l"(key), "l"(aux), "l"(s)
        : "memory");
    if (got_k == old_k && got_a == old_a) return;    // swapped in
    old_k = got_k;
    old_a = got_a;
    if (key <= old_k) return;                         // someone better is already there
  }
}

// Rare path of the epilogue, kept out of line so that the 32-fold unrolled epilogue stays small (at p = 1
// it runs on every 8 KB row and must not thrash the instruction cache).
__device__ __noinline__ void emit_candidate(Slot* slots_t, unsigned j, float rho2, float chi, float thresh, int log_w) {
  const float rho = sqrtf(rho2);
  if (rho > thresh)
    slot_max(slots_t + (j >> log_w), ((unsigned long long)__float_as_uint(rho) << 32) | (unsigned long long)(0xFFFFFFFFu - j),
             (unsigned long long)__float_as_uint(chi));
}

__device__ __forceinline__ float2 cis_frac_p2(unsigned num, int log_n) {
  // e^{2 pi i num / 2^log_n}; num is reduced mod 2^log_n first so that 2 num / n is exact in fp32
  num &= (1u << log_n) - 1u;
  float s, c;
  sincospif(2.0f * (float)num / (float)(1u << log_n), &s, &c);
  return make_float2(c, s);
}

// ---- TMA (bulk async copy) + mbarrier helpers --------------------------------------------------------
__device__ __forceinline__ unsigned smem_u32(const void* p) { return (unsigned)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void mbar_init(unsigned long long* bar, unsigned count) {
  asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(bar)), "r"(count) : "memory");
}
__device__ __forceinline__ void mbar_expect_tx(unsigned long long* bar, unsigned bytes) {
  asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(bar)), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_wait(unsigned long long* bar, unsigned parity) {
  unsigned ok;
  do {
    asm volatile(
        "{\n\t.reg .pred p;\n\t"
        "mbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n\t"
        "selp.u32 %0, 1, 0, p;\n\t}"
        : "=r"(ok)
        : "r"(smem_u32(bar)), "r"(parity)
        : "memory");
  } while (!ok);
}
// one contiguous row global -> shared, completion signalled on the mbarrier (SASS: UBLKCP)
__device__ __forceinline__ void bulk_load_row(void* dst, const void* src, unsigned bytes, unsigned long long* bar,
                                              unsigned long long policy) {
  asm volatile(
      "cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes.L2::cache_hint [%0], [%1], %2, [%3], %4;" ::"r"(
          smem_u32(dst)),
      "l"(src), "r"(bytes), "r"(smem_u32(bar)), "l"(policy)
      : "memory");
}

// one row (ja, jb) of a slot of the decimated path's band buffer [slot][ja][c][jb][jm]: 32 pieces of 256 B, 8 KB apart,
// gathered by ONE tensor copy (box {jm: 256 B, jb: 1, c: 32, tile: 1}); lands as [c][256 B] (SASS: UTMALDG)
__device__ __forceinline__ void tensor_load_row(void* dst, const CUtensorMap* tmap, int jb, int tile, unsigned long long* bar,
                                                unsigned long long policy) {
  asm volatile(
      "cp.async.bulk.tensor.4d.shared::cluster.global.mbarrier::complete_tx::bytes.L2::cache_hint [%0], [%1, {%2, %3, %4, %5}], [%6], %7;" ::"r"(
          smem_u32(dst)),
      "l"(tmap), "r"(0), "r"(jb), "r"(0), "r"(tile), "r"(smem_u32(bar)), "l"(policy)
      : "memory");
}

constexpr int kRowBytes = kN2 * (int)sizeof(float2);      // 8 KB
constexpr int kP2Ring = 3;                                // row buffers per warp

// Shared memory: [twiddles 32x32][warp 0: ring of kP2Ring rows][warp 1: ...]...[mbarriers, kP2Ring per warp].
template <bool STORE, bool SERIES>
__global__ void __launch_bounds__(kP2Warps * 32, 1) k_pass2(P2Args a) {
  extern __shared__ __align__(128) float2 smem2[];
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  float2* tw_s = smem2;                                               // [c][jm]
  float2* bufs = smem2 + 1024 + warp * (kP2Ring * kN2);
  unsigned long long* bars = reinterpret_cast<unsigned long long*>(smem2 + 1024 + kP2Warps * kP2Ring * kN2) + kP2Ring * warp;
  for (int i = threadIdx.x; i < 1024; i += blockDim.x) tw_s[i] = a.tw_p2[i];
  __syncthreads();                                                    // the only CTA-wide barrier

  const int p = a.p;
  const int total_warps = gridDim.x * kP2Warps;
  const int first_row = blockIdx.x * kP2Warps + warp;
  if (first_row >= a.n_rows) return;                                  // warps are independent: no CTA barrier below
  const int my_rows = (a.n_rows - first_row + total_warps - 1) / total_warps;
  const int n_items = my_rows * p;                                    // (row, band) pairs, band fastest
  const size_t band_stride = (size_t)a.n1 * kN2;
  const int n1_mask = a.n1 - 1;

  unsigned long long policy;
  asm volatile("createpolicy.fractional.L2::evict_first.b64 %0, 1.0;" : "=l"(policy));

  // prefetch cursor (next item to request)
  // Rows are walked from the END of the band buffer: what pass 1 wrote last is still in L2.
  const int last_row = a.n_rows - 1 - first_row;
  int pf_item = 0, pf_l = 0, pf_row = last_row;
  auto prefetch = [&]() {
    // caller: lane 0 only, and only after every lane has consumed the buffer being refilled
    const int tb = pf_row >> a.log_n1, j1 = pf_row & n1_mask;
    const float2* src = a.y + ((size_t)(tb * p + pf_l) * a.n1 + j1) * kN2;
    const int b = pf_item % kP2Ring;
    asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
    mbar_expect_tx(&bars[b], kRowBytes);
    bulk_load_row(bufs + b * kN2, src, kRowBytes, &bars[b], policy);
  };
  auto advance = [&]() {
    ++pf_item;
    if (++pf_l == p) { pf_l = 0; pf_row -= total_warps; }
  };
  if (lane == 0) {
#pragma unroll
    for (int b = 0; b < kP2Ring; ++b) mbar_init(&bars[b], 1);
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
  }
  __syncwarp();
#pragma unroll 1
  for (int b = 0; b < kP2Ring && pf_item < n_items; ++b) {
    if (lane == 0) prefetch();
    advance();
  }

  float2 az[32];
  float aq[32];
#pragma unroll
  for (int i = 0; i < 32; ++i) { az[i] = make_float2(0.f, 0.f); aq[i] = 0.f; }

  int l = 0, row = last_row;
#pragma unroll 1
  for (int item = 0; item < n_items; ++item) {
    const int b = item % kP2Ring;
    const float2* cur = bufs + b * kN2;
    mbar_wait(&bars[b], (item / kP2Ring) & 1);
    float2 x[32];
#pragma unroll
    for (int c = 0; c < 32; ++c) x[brev<32>(c)] = cmul(cur[32 * c + lane], tw_s[32 * c + lane]);     // lane = jm
    fft_dit<32>(x);                                                       // over c -> jc; j2 = lane + 32 jc
    __syncwarp();                                                         // every lane holds its 32 values
    if (pf_item < n_items) {
      if (lane == 0) prefetch();
      advance();
    }
    if constexpr (STORE) {
#pragma unroll
      for (int jc = 0; jc < 32; ++jc)
        a.dense_out[(size_t)row + ((size_t)(lane + 32 * jc) << a.log_n1)] = x[jc];
      row -= total_warps;
    } else {
#pragma unroll
      for (int jc = 0; jc < 32; ++jc) {
        const float2 z = x[jc];
        az[jc] = cadd(az[jc], z);
        aq[jc] = fmaf(z.x, z.x, fmaf(z.y, z.y, aq[jc]));
      }
      if (++l == p) {
        // ---- epilogue of one row: rho, chi^2 and the trigger slots (steps a4, a5) ----
        const int tb = row >> a.log_n1, j1 = row & n1_mask;
        const float scale = __ldg(&a.meta[tb].scale_rho2);
        const float fp_scale = (float)p * scale, inv_p = 1.0f / (float)p;
        const float thr2 = a.thresh * a.thresh * 0.999f;
        Slot* slots_t = a.slots ? a.slots + (size_t)tb * a.n_windows : nullptr;
#pragma unroll
        for (int jc = 0; jc < 32; ++jc) {
          const float z2 = fmaf(az[jc].x, az[jc].x, az[jc].y * az[jc].y);
          const float rho2 = z2 * scale;                                        // Eq. 3 squared
          const float chi = fmaxf(aq[jc] - z2 * inv_p, 0.f) * fp_scale;         // Eq. 5
          const unsigned j = (unsigned)j1 + ((unsigned)(lane + 32 * jc) << a.log_n1);
          if constexpr (SERIES) {
            if (a.series_rho) a.series_rho[j] = sqrtf(rho2);
            if (a.series_chi) a.series_chi[j] = chi;
          }
          if (rho2 > thr2 && slots_t) emit_candidate(slots_t, j, rho2, chi, a.thresh, a.log_w);
          az[jc] = make_float2(0.f, 0.f);
          aq[jc] = 0.f;
        }
        l = 0;
        row -= total_warps;
      }
    }
  }
}

// ---------------------------------------------------------------------------------------------------
// Decimated path: the same last stage and epilogue over a template's EFFECTIVE bands (gwmf_internal.cuh).  A row
// (template, j1) owns n_eff 8 KB rows of the band buffer, at slots eff_prefix - slot_base + e:
//     Z (e = 0): z  += x                      the narrow bands' share of z, one transform for all of them
//     U (e = 1): q  += Re x                   sum over the narrow bands of |z_l|^2 (bandpower.cu)
//     D (wide) : z  += x,  q += |x|^2         a wide band's own transform, as in k_pass2
// then the same rho / chi^2 / trigger epilogue.  Warps are persistent and prefetch through the same ring of TMA
// bulk copies, across band and row boundaries.
// ---------------------------------------------------------------------------------------------------
struct P2EArgs {
  P2Args b;                   // b.meta: first template of the (pair-aligned) batch; b.n_rows: rows of [t_begin, t_begin + count)
  int slot_base;              // eff_prefix of the first template of the batch
  int log_na;                 // log2(n1 / 32): j1 = ja + NA jb
  int batch;                  // templates of the batch (spectra and pass 1 were run for all of them)
  int t_begin;                // first template of the batch whose rows this launch processes (batch-relative)
};

// SINGLE: every template of the launch has exactly one effective band (p = 1, or chi^2 on demand): z is that band's
// transform, no sums over bands are kept, and the epilogue is one compare of |z|^2 against the threshold per sample
// (chi^2 is 0 by definition for p = 1 and is filled in later by k_chisq_at in the on-demand mode).
constexpr int kP2EWarps = 12;    // k_pass2_eff: 12 warps per SM with a ring of 2 rows each (192 KB): the kernel is bound by the
constexpr int kP2ERing = 2;     // latency of its per-row chains, not by HBM, once a template needs ~2 transforms

template <bool SERIES, bool SINGLE>
__global__ void __launch_bounds__(kP2EWarps * 32, 1) k_pass2_eff(P2EArgs ea, const __grid_constant__ CUtensorMap tmap) {
  const P2Args& a = ea.b;
  extern __shared__ __align__(128) float2 smem2[];
  __shared__ int s_slot0[kMaxBatch + 2];      // first slot of template tb (batch-relative)
  __shared__ int s_neff[kMaxBatch + 2];       // rows to read | has_s << 8 | guest of a pair << 9
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  float2* tw_s = smem2;                                               // [c][jm]
  float2* bufs = smem2 + 1024 + warp * (kP2ERing * kN2);
  unsigned long long* bars = reinterpret_cast<unsigned long long*>(smem2 + 1024 + kP2EWarps * kP2ERing * kN2) + kP2ERing * warp;
  for (int i = threadIdx.x; i < 1024; i += blockDim.x) tw_s[i] = a.tw_p2[i];
  for (int t = threadIdx.x; t < ea.batch; t += blockDim.x) {
    s_slot0[t] = a.meta[t].eff_prefix - ea.slot_base;
    const bool guest = a.meta[t].pair == 2;     // reads one row more than it owns: the pair band of template t - 1
    s_neff[t] = (a.meta[t].n_eff + (guest ? 1 : 0)) | (a.meta[t].s_mask ? 256 : 0) | (guest ? 512 : 0);
  }
  __syncthreads();                                                    // the only CTA-wide barrier

  const int total_warps = gridDim.x * kP2EWarps;
  const int first_row = blockIdx.x * kP2EWarps + warp;
  if (first_row >= a.n_rows) return;                                  // warps are independent: no CTA barrier below
  const int n1_mask = a.n1 - 1;

  unsigned long long policy, policy_keep;
  asm volatile("createpolicy.fractional.L2::evict_first.b64 %0, 1.0;" : "=l"(policy));
  // a pair band is read twice, by the guest's row first (rows are walked downwards) and about one row-time later by
  // its owner's: the first read keeps it in L2, the second one releases it
  asm volatile("createpolicy.fractional.L2::evict_last.b64 %0, 1.0;" : "=l"(policy_keep));

  // Rows are walked from the END of the band buffer: what pass 1 wrote last is still in L2.
  const int last_row = a.n_rows - 1 - first_row;
  int pf_item = 0, pf_e = 0, pf_row = last_row;                       // prefetch cursor (next item to request)
  auto prefetch = [&]() {
    // caller: lane 0 only, and only after every lane has consumed the buffer being refilled
    const int tb = ea.t_begin + (pf_row >> a.log_n1), j1 = pf_row & n1_mask;
    // item e of a row -> slot: a guest's item 1 is the pair band of its owner (slot 1 of template tb - 1)
    const int slot = (s_neff[tb] & 512) ? (pf_e == 1 ? s_slot0[tb - 1] + 1 : s_slot0[tb] + pf_e - (pf_e > 1 ? 1 : 0))
                                        : s_slot0[tb] + pf_e;
    const int b = pf_item % kP2ERing;
    asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
    mbar_expect_tx(&bars[b], kRowBytes);
    // j1 = ja + NA jb: tile (slot, ja), row jb of each of its 32 pieces
    tensor_load_row(bufs + b * kN2, &tmap, j1 >> ea.log_na, (slot << ea.log_na) + (j1 & ((1 << ea.log_na) - 1)), &bars[b],
                    ((s_neff[tb] & 512) && pf_e == 1) ? policy_keep : policy);
  };
  auto advance = [&]() {
    ++pf_item;
    if (++pf_e == (s_neff[ea.t_begin + (pf_row >> a.log_n1)] & 255)) { pf_e = 0; pf_row -= total_warps; }
  };
  if (lane == 0) {
#pragma unroll
    for (int b = 0; b < kP2ERing; ++b) mbar_init(&bars[b], 1);
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
  }
  __syncwarp();
#pragma unroll 1
  for (int b = 0; b < kP2ERing && pf_row >= 0; ++b) {
    if (lane == 0) prefetch();
    advance();
  }

  float2 az[32];
  float aq[32];
#pragma unroll
  for (int i = 0; i < 32; ++i) { az[i] = make_float2(0.f, 0.f); aq[i] = 0.f; }

  int item = 0;
#pragma unroll 1
  for (int row = last_row; row >= 0; row -= total_warps) {
    const int tb = ea.t_begin + (row >> a.log_n1), j1 = row & n1_mask;
    const int ne = s_neff[tb] & 255;
    const bool has_s = (s_neff[tb] & 256) != 0, guest = (s_neff[tb] & 512) != 0;
#pragma unroll 1
    for (int e = 0; e < ne; ++e, ++item) {
      const int b = item % kP2ERing;
      const float2* cur = bufs + b * kN2;
      mbar_wait(&bars[b], (item / kP2ERing) & 1);
      float2 x[32];
#pragma unroll
      // pass 1 stores the 16-byte chunk ch of a 256 B piece at chunk ch ^ (jb & 15)
      const int sl = lane ^ (((j1 >> ea.log_na) & 15) << 1);
      for (int c = 0; c < 32; ++c) {                                        // lane = jm
        x[brev<32>(c)] = cmul(cur[32 * c + sl], tw_s[32 * c + lane]);
      }
      fft_dit<32>(x);                                                       // over c -> jc; j2 = lane + 32 jc
      __syncwarp();                                                         // every lane holds its 32 values
      if (pf_row >= 0) {
        if (lane == 0) prefetch();
        advance();
      }
      if constexpr (SINGLE) {
        // ---- the row's only band: epilogue straight from the transform (steps a4, a5 without chi^2) ----
        const float scale = __ldg(&a.meta[tb].scale_rho2);
        const float thr_z2 = a.thresh * a.thresh * 0.999f / scale;            // rho^2 > thr^2  <=>  |z|^2 > thr^2 / scale
        Slot* slots_t = a.slots ? a.slots + (size_t)tb * a.n_windows : nullptr;
        if constexpr (SERIES) {
#pragma unroll
          for (int jc = 0; jc < 32; ++jc) {
            const float z2 = fmaf(x[jc].x, x[jc].x, x[jc].y * x[jc].y);
            const unsigned j = (unsigned)j1 + ((unsigned)(lane + 32 * jc) << a.log_n1);
            if (a.series_rho) a.series_rho[j] = sqrtf(z2 * scale);
            if (a.series_chi) a.series_chi[j] = 0.f;
            if (z2 > thr_z2 && slots_t) emit_candidate(slots_t, j, z2 * scale, 0.f, a.thresh, a.log_w);
          }
        } else {
          // events are rare: one running maximum per lane, the per-sample test only where it crosses
          float zmax = 0.f;
#pragma unroll
          for (int jc = 0; jc < 32; ++jc) zmax = fmaxf(zmax, fmaf(x[jc].x, x[jc].x, x[jc].y * x[jc].y));
          if (zmax > thr_z2 && slots_t) {
#pragma unroll
            for (int jc = 0; jc < 32; ++jc) {
              const float z2 = fmaf(x[jc].x, x[jc].x, x[jc].y * x[jc].y);
              if (z2 > thr_z2)
                emit_candidate(slots_t, (unsigned)j1 + ((unsigned)(lane + 32 * jc) << a.log_n1), z2 * scale, 0.f, a.thresh, a.log_w);
            }
          }
        }
        continue;
      }
      if (has_s && e == 0) {                    // Z
#pragma unroll
        for (int jc = 0; jc < 32; ++jc) az[jc] = cadd(az[jc], x[jc]);
      } else if (has_s && e == 1) {             // U: real part; the guest of a pair owns the imaginary part
        if (guest) {
#pragma unroll
          for (int jc = 0; jc < 32; ++jc) aq[jc] += x[jc].y;
        } else {
#pragma unroll
          for (int jc = 0; jc < 32; ++jc) aq[jc] += x[jc].x;
        }
      } else {                                  // D
#pragma unroll
        for (int jc = 0; jc < 32; ++jc) {
          const float2 z = x[jc];
          az[jc] = cadd(az[jc], z);
          aq[jc] = fmaf(z.x, z.x, fmaf(z.y, z.y, aq[jc]));
        }
      }
    }
    if constexpr (SINGLE) continue;
    // ---- epilogue of one row: rho, chi^2 and the trigger slots (steps a4, a5) ----
    const float scale = __ldg(&a.meta[tb].scale_rho2);
    const float fp_scale = (float)a.p * scale, inv_p = 1.0f / (float)a.p;
    const float thr2 = a.thresh * a.thresh * 0.999f;
    Slot* slots_t = a.slots ? a.slots + (size_t)tb * a.n_windows : nullptr;
    if constexpr (SERIES) {
#pragma unroll
      for (int jc = 0; jc < 32; ++jc) {
        const float z2 = fmaf(az[jc].x, az[jc].x, az[jc].y * az[jc].y);
        const float rho2 = z2 * scale;                                        // Eq. 3 squared
        const float chi = fmaxf(aq[jc] - z2 * inv_p, 0.f) * fp_scale;         // Eq. 5
        const unsigned j = (unsigned)j1 + ((unsigned)(lane + 32 * jc) << a.log_n1);
        if (a.series_rho) a.series_rho[j] = sqrtf(rho2);
        if (a.series_chi) a.series_chi[j] = chi;
        if (rho2 > thr2 && slots_t) emit_candidate(slots_t, j, rho2, chi, a.thresh, a.log_w);
      }
    } else {
      // events are rare: one running maximum of |z|^2 per lane; rho, chi^2 and the slot update only where it crosses
      float zmax = 0.f;
#pragma unroll
      for (int jc = 0; jc < 32; ++jc) zmax = fmaxf(zmax, fmaf(az[jc].x, az[jc].x, az[jc].y * az[jc].y));
      if (zmax * scale > thr2 && slots_t) {
#pragma unroll
        for (int jc = 0; jc < 32; ++jc) {
          const float z2 = fmaf(az[jc].x, az[jc].x, az[jc].y * az[jc].y);
          const float rho2 = z2 * scale;                                      // Eq. 3 squared
          if (rho2 > thr2) {
            const float chi = fmaxf(aq[jc] - z2 * inv_p, 0.f) * fp_scale;     // Eq. 5
            emit_candidate(slots_t, (unsigned)j1 + ((unsigned)(lane + 32 * jc) << a.log_n1), rho2, chi, a.thresh, a.log_w);
          }
        }
      }
    }
#pragma unroll
    for (int jc = 0; jc < 32; ++jc) { az[jc] = make_float2(0.f, 0.f); aq[jc] = 0.f; }
  }
}

// ---------------------------------------------------------------------------------------------------
// Spill-free path (the library's choice for n <= 2^20; gwmf_uses_fused): narrow bands never reach HBM.  A CTA
// owns 8 consecutive rows j1 of one template (one per warp) and walks the p bands.  For a narrow band (<= 32
// input rows) the row of Y is formed directly from the correlated spectrum,
//     Y_l[j1][k2] = e^{2 pi i j1 k2/n} sum_i Q[1024 k1_i + k2] e^{2 pi i j1 k1_i/n1}
// (R complex MACs per sample with row-constant twiddles).  The band's rows come from the band-separated copy
// of the correlated spectrum (k_correlate_bands: rows of a band contiguous, bins outside the band zeroed) by
// one TMA bulk copy per chunk of <= 8 rows, double-buffered in shared memory, issued one chunk ahead; one CTA
// barrier per chunk hands the buffer over.  Both 32-point stages of the row transform then run in the warp
// (transpose through its padded tile), followed by the accumulation and epilogue of k_pass2.  Wide bands come
// from the band buffer (generic pass-1 kernel + row stage) through a TMA load, as in k_pass2.
// ---------------------------------------------------------------------------------------------------
struct FArgs {
  P2Args b;
  const float2* qb;           // [batch][rows_cap][1024] band-separated correlated spectra (k_correlate_bands)
  const float2* tw_n1;        // e^{2 pi i m/n1}
  int log_n;
  int n_groups;               // batch * n1 / 8
  int rows_cap;
};

constexpr int kFRows = 8;                       // input rows staged per chunk (64 KB)
constexpr int kFTile = 32 * 33;                 // per-warp tile (float2): padded transpose tile / TMA landing buffer

template <bool SERIES>
__global__ void __launch_bounds__(256, 1) k_fused(FArgs fa) {
  const P2Args& a = fa.b;
  extern __shared__ __align__(128) float2 smem2[];
  float2* tw_s = smem2;                                   // [c][jm] e^{2 pi i c jm/1024}
  float2* Qs = smem2 + 1024;                              // [2][kFRows][1024]: double-buffered chunk of band rows
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  float2* buf = Qs + 2 * kFRows * 1024 + warp * kFTile;
  float2* beta = Qs + 2 * kFRows * 1024 + 8 * kFTile + warp * 32;
  unsigned long long* bars = reinterpret_cast<unsigned long long*>(Qs + 2 * kFRows * 1024 + 8 * kFTile + 8 * 32);
  unsigned long long* bar = bars + warp;                  // this warp's TMA barrier (wide bands)
  unsigned long long* full = bars + 8;                    // full[2]: chunk landed in Qs[b]
  int* s_meta = reinterpret_cast<int*>(bars + 10);        // [0..33): edges, [40..74): row_off
  for (int i = tid; i < 1024; i += 256) tw_s[i] = a.tw_p2[i];
  if (lane == 0) mbar_init(bar, 1);
  if (tid == 0) { mbar_init(&full[0], 1); mbar_init(&full[1], 1); }
  asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
  __syncthreads();
  unsigned long long policy;
  asm volatile("createpolicy.fractional.L2::evict_first.b64 %0, 1.0;" : "=l"(policy));

  const int p = a.p;
  const int n1 = a.n1, n1m = n1 - 1;
  const int groups_per_t = n1 >> 3;
  unsigned tma_phase = 0;           // uses of this warp's barrier
  unsigned use0 = 0, use1 = 0;      // uses of full[0], full[1] (uniform over the CTA)
  int cidx = 0;                     // chunks consumed so far (buffer = cidx & 1)

#pragma unroll 1
  for (int g = blockIdx.x; g < fa.n_groups; g += gridDim.x) {
    const int tb = g / groups_per_t, j1 = ((g - tb * groups_per_t) << 3) + warp;
    const TemplateMeta* mt = a.meta + tb;
    __syncthreads();                                       // s_meta and both chunk buffers are free
    if (tid <= p) { s_meta[tid] = mt->edges[tid]; s_meta[40 + tid] = mt->row_off[tid]; }
    const unsigned wide_mask = mt->wide_mask;
    const float2* qb_t = fa.qb + (size_t)tb * fa.rows_cap * kN2;
    // row twiddles: e^{2 pi i j1 k2/n} = alpha_lane * beta^m with k2 = 32 m + lane
    beta[lane] = cis_frac_p2(((unsigned)j1 * 32u * (unsigned)lane), fa.log_n);
    const float2 alpha = cis_frac_p2((unsigned)j1 * (unsigned)lane, fa.log_n);
    __syncthreads();
    // chunk (l, r0) of the narrow bands: rows row_off[l] + r0 .. of Qb; issue() starts its bulk copy into Qs[b]
    auto issue = [&](int l, int r0, int b) {
      const int R = s_meta[40 + l + 1] - s_meta[40 + l];
      const int rc = R - r0 < kFRows ? R - r0 : kFRows;
      const unsigned bytes = (unsigned)rc * kN2 * (unsigned)sizeof(float2);
      asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
      mbar_expect_tx(&full[b], bytes);
      bulk_load_row(Qs + b * kFRows * 1024, qb_t + (size_t)(s_meta[40 + l] + r0) * kN2, bytes, &full[b], policy);
    };
    auto next_chunk = [&](int& l, int& r0) -> bool {       // advance to the following chunk of this group
      const int R = s_meta[40 + l + 1] - s_meta[40 + l];
      if (r0 + kFRows < R) { r0 += kFRows; return true; }
      for (int l2 = l + 1; l2 < p; ++l2)
        if (s_meta[40 + l2 + 1] > s_meta[40 + l2]) { l = l2; r0 = 0; return true; }
      return false;
    };
    {   // first chunk of the group
      int l0 = -1;
      for (int l2 = 0; l2 < p; ++l2)
        if (s_meta[40 + l2 + 1] > s_meta[40 + l2]) { l0 = l2; break; }
      if (l0 >= 0 && tid == 0) issue(l0, 0, cidx & 1);
    }

    float2 az[32];
    float aq[32];
#pragma unroll
    for (int i = 0; i < 32; ++i) { az[i] = make_float2(0.f, 0.f); aq[i] = 0.f; }

#pragma unroll 1
    for (int l = 0; l < p; ++l) {
      float2 x[32];
      if ((wide_mask >> l) & 1u) {
        // wide band: the A row was written by the generic pass-1 kernel + row stage
        const float2* src = a.y + ((size_t)(tb * p + l) * n1 + j1) * kN2;
        if (lane == 0) {
          asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
          mbar_expect_tx(bar, kN2 * (unsigned)sizeof(float2));
          bulk_load_row(buf, src, kN2 * (unsigned)sizeof(float2), bar, policy);
        }
        mbar_wait(bar, tma_phase & 1u);
        ++tma_phase;
#pragma unroll
        for (int c = 0; c < 32; ++c) x[brev<32>(c)] = cmul(buf[32 * c + lane], tw_s[32 * c + lane]);
        __syncwarp();
      } else {
        const int R = s_meta[40 + l + 1] - s_meta[40 + l];
        if (R == 0) continue;                          // empty band: z_l = 0
        const int e_lo = s_meta[l], e_hi = s_meta[l + 1];
        const int row_lo = e_lo >> kLogN2, row_hi = (e_hi - 1) >> kLogN2;
        float2 acc[32];
#pragma unroll
        for (int m = 0; m < 32; ++m) acc[m] = make_float2(0.f, 0.f);
#pragma unroll 1
        for (int r0 = 0; r0 < R; r0 += kFRows) {
          const int rc = R - r0 < kFRows ? R - r0 : kFRows;
          const int b = cidx & 1;
          __syncthreads();                             // every warp is done with the chunk that used Qs[b ^ 1]
          if (tid == 0) {
            int ln = l, rn = r0;
            if (next_chunk(ln, rn)) issue(ln, rn, b ^ 1);
          }
          mbar_wait(&full[b], (b ? use1 : use0) & 1u);
          if (b) ++use1; else ++use0;
          ++cidx;
          const float2* qbase = Qs + b * kFRows * 1024 + lane;
#pragma unroll 1
          for (int i = 0; i < rc; ++i) {
            const int k1 = row_lo + r0 + i;
            const tw4 r = make_tw4(cmul(fa.tw_n1[(j1 * k1) & n1m], alpha));   // e^{2 pi i j1 (k1/n1 + lane/n)}
            const float2* qs = qbase + i * 1024;
            // the band's first and last row are only partly inside it: skip the blocks of 8 m (256 bins) that
            // hold nothing but zeros (warp-uniform branches)
            const int m_lo = (k1 == row_lo) ? ((e_lo & 1023) >> 5) : 0;
            const int m_hi = (k1 == row_hi) ? (((e_hi - 1) & 1023) >> 5) + 1 : 32;
#pragma unroll
            for (int mb = 0; mb < 4; ++mb) {
              if (8 * mb + 7 >= m_lo && 8 * mb < m_hi) {
#pragma unroll
                for (int m = 8 * mb; m < 8 * mb + 8; ++m) {
                  const float2 qv = qs[32 * m];
                  acc[m] = unpk(fma2(pk(-qv.y, qv.x), r.yy, fma2(pk(qv), r.xx, pk(acc[m]))));
                }
              }
            }
          }
        }
        // first row stage (over m), lane = c
#pragma unroll
        for (int m = 0; m < 32; ++m) x[brev<32>(m)] = cmul(acc[m], beta[m]);
        fft_dit<32>(x);
#pragma unroll
        for (int jm = 0; jm < 32; ++jm) buf[lane * 33 + jm] = x[jm];
        __syncwarp();
#pragma unroll
        for (int c = 0; c < 32; ++c) x[brev<32>(c)] = cmul(buf[c * 33 + lane], tw_s[32 * c + lane]);   // lane = jm
        __syncwarp();
      }
      fft_dit<32>(x);                                   // over c -> jc
#pragma unroll
      for (int jc = 0; jc < 32; ++jc) {
        const float2 z = x[jc];
        az[jc] = cadd(az[jc], z);
        aq[jc] = fmaf(z.x, z.x, fmaf(z.y, z.y, aq[jc]));
      }
    }
    // ---- epilogue of one row: rho, chi^2 and the trigger slots (steps a4, a5) ----
    {
      const float scale = mt->scale_rho2;
      const float fp_scale = (float)p * scale, inv_p = 1.0f / (float)p;
      const float thr2 = a.thresh * a.thresh * 0.999f;
      Slot* slots_t = a.slots ? a.slots + (size_t)tb * a.n_windows : nullptr;
#pragma unroll
      for (int jc = 0; jc < 32; ++jc) {
        const float z2 = fmaf(az[jc].x, az[jc].x, az[jc].y * az[jc].y);
        const float rho2 = z2 * scale;                                        // Eq. 3 squared
        const float chi = fmaxf(aq[jc] - z2 * inv_p, 0.f) * fp_scale;         // Eq. 5
        const unsigned j = (unsigned)j1 + ((unsigned)(lane + 32 * jc) << a.log_n1);
        if constexpr (SERIES) {
          if (a.series_rho) a.series_rho[j] = sqrtf(rho2);
          if (a.series_chi) a.series_chi[j] = chi;
        }
        if (rho2 > thr2 && slots_t) emit_candidate(slots_t, j, rho2, chi, a.thresh, a.log_w);
      }
    }
  }
}

constexpr size_t kFusedSmem = (size_t)(1024 + 2 * kFRows * 1024 + 8 * kFTile + 8 * 32) * sizeof(float2) +
                              10 * sizeof(unsigned long long) + 80 * sizeof(int);

cudaError_t launch_fused_filter(Ctx* c, int first, int count, int parity, bool update_slots, float* series_rho, float* series_chi) {
  FArgs fa;
  P2Args& a = fa.b;
  a.y = ws_ptr<float2>(c, c->lay.y);
  a.tw_p2 = ws_ptr<float2>(c, c->lay.tw_p2);
  a.meta = ws_ptr<TemplateMeta>(c, c->lay.meta) + first;
  a.slots = update_slots ? ws_ptr<Slot>(c, c->lay.slots) + (size_t)first * c->n_windows : nullptr;
  a.series_rho = series_rho;
  a.series_chi = series_chi;
  a.dense_out = nullptr;
  a.p = c->prm.p;
  a.n1 = c->n1;
  a.log_n1 = c->log_n - kLogN2;
  int lw = 0;
  while ((1 << lw) < c->prm.window) ++lw;
  a.log_w = lw;
  a.n_windows = c->n_windows;
  a.n_rows = count * c->n1;
  a.thresh = (float)c->prm.rho_thresh;
  fa.rows_cap = qb_rows_cap(c);
  fa.qb = ws_ptr<float2>(c, c->lay.qb) + (size_t)parity * c->lay.batch * fa.rows_cap * kN2;
  fa.tw_n1 = ws_ptr<float2>(c, c->lay.tw_n1);
  fa.log_n = c->log_n;
  fa.n_groups = count * (c->n1 / 8);
  const int grid = fa.n_groups < c->n_sms ? fa.n_groups : c->n_sms;
  if (series_rho || series_chi) k_fused<true><<<grid, 256, kFusedSmem, c->stream>>>(fa);
  else k_fused<false><<<grid, 256, kFusedSmem, c->stream>>>(fa);
  c->launches++;
  return cudaGetLastError();
}

constexpr size_t kP2Smem = (size_t)(1024 + kP2Warps * kP2Ring * kN2) * sizeof(float2) + kP2Warps * kP2Ring * sizeof(unsigned long long);
constexpr size_t kP2ESmem = (size_t)(1024 + kP2EWarps * kP2ERing * kN2) * sizeof(float2) + kP2EWarps * kP2ERing * sizeof(unsigned long long);

// Opt-in to > 48 KB of dynamic shared memory on the CURRENT device (gwmf_create calls this for every context).
cudaError_t configure_pass2() {
  cudaError_t e = cudaFuncSetAttribute(k_pass2<false, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)kP2Smem);
  if (e == cudaSuccess) e = cudaFuncSetAttribute(k_pass2<false, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)kP2Smem);
  if (e == cudaSuccess) e = cudaFuncSetAttribute(k_pass2<true, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)kP2Smem);
  if (e == cudaSuccess) e = cudaFuncSetAttribute(k_pass2_eff<false, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)kP2ESmem);
  if (e == cudaSuccess) e = cudaFuncSetAttribute(k_pass2_eff<true, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)kP2ESmem);
  if (e == cudaSuccess) e = cudaFuncSetAttribute(k_pass2_eff<false, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)kP2ESmem);
  if (e == cudaSuccess) e = cudaFuncSetAttribute(k_pass2_eff<true, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)kP2ESmem);
  if (e == cudaSuccess) e = cudaFuncSetAttribute(k_fused<false>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)kFusedSmem);
  if (e == cudaSuccess) e = cudaFuncSetAttribute(k_fused<true>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)kFusedSmem);
  return e;
}

// The band buffer of the decimated path as a tensor of fp32: dims (fastest first) {64 floats = 32 jm, 32 jb, 32 c,
// tiles = y_slots * NA}; pass 2 fetches row (ja, jb) of a slot with the box {64, 1, 32, 1} = 8 KB.  cuTensorMapEncodeTiled
// is fetched from the driver at run time (no libcuda at link time).
cudaError_t make_band_tensor_map(Ctx* c) {
  typedef CUresult (*EncodeFn)(CUtensorMap*, CUtensorMapDataType, cuuint32_t, void*, const cuuint64_t*, const cuuint64_t*,
                               const cuuint32_t*, const cuuint32_t*, CUtensorMapInterleave, CUtensorMapSwizzle,
                               CUtensorMapL2promotion, CUtensorMapFloatOOBfill);
  void* fn = nullptr;
  cudaDriverEntryPointQueryResult qres;
  cudaError_t e = cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &fn, cudaEnableDefault, &qres);
  if (e != cudaSuccess) return e;
  if (!fn || qres != cudaDriverEntryPointSuccess) return cudaErrorNotSupported;
  const int na = c->n1 / 32;
  if (na < 1) { memset(&c->band_tmap, 0, sizeof(c->band_tmap)); return cudaSuccess; }     // n = 2^14 never takes this path
  const cuuint64_t dims[4] = {64, 32, 32, (cuuint64_t)c->lay.y_slots * (cuuint64_t)na};
  const cuuint64_t strides[3] = {256, 8192, 262144};                                       // bytes, dims 1..3
  const cuuint32_t box[4] = {64, 1, 32, 1};
  const cuuint32_t estr[4] = {1, 1, 1, 1};
  const CUresult r = reinterpret_cast<EncodeFn>(fn)(&c->band_tmap, CU_TENSOR_MAP_DATA_TYPE_FLOAT32, 4, c->ws + c->lay.y, dims, strides,
                                                    box, estr, CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_NONE,
                                                    CU_TENSOR_MAP_L2_PROMOTION_L2_256B, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
  return r == CUDA_SUCCESS ? cudaSuccess : cudaErrorInvalidValue;
}

static int p2_grid(const Ctx* c, int n_rows) {
  const int want = (n_rows + kP2Warps - 1) / kP2Warps;
  return want < c->n_sms ? want : c->n_sms;               // persistent: at most one CTA per SM
}

cudaError_t launch_pass2_filter(Ctx* c, int first, int count, bool update_slots, float* series_rho, float* series_chi) {
  P2Args a;
  a.y = ws_ptr<float2>(c, c->lay.y);
  a.tw_p2 = ws_ptr<float2>(c, c->lay.tw_p2);
  a.meta = ws_ptr<TemplateMeta>(c, c->lay.meta) + first;
  a.slots = update_slots ? ws_ptr<Slot>(c, c->lay.slots) + (size_t)first * c->n_windows : nullptr;
  a.series_rho = series_rho;
  a.series_chi = series_chi;
  a.dense_out = nullptr;
  a.p = c->prm.p;
  a.n1 = c->n1;
  a.log_n1 = c->log_n - kLogN2;
  int lw = 0;
  while ((1 << lw) < c->prm.window) ++lw;
  a.log_w = lw;
  a.n_windows = c->n_windows;
  a.n_rows = count * c->n1;
  a.thresh = (float)c->prm.rho_thresh;
  if (series_rho || series_chi) k_pass2<false, true><<<p2_grid(c, a.n_rows), kP2Warps * 32, kP2Smem, c->stream>>>(a);
  else k_pass2<false, false><<<p2_grid(c, a.n_rows), kP2Warps * 32, kP2Smem, c->stream>>>(a);
  c->launches++;
  return cudaGetLastError();
}

cudaError_t launch_pass2_dense(Ctx* c, const float2* d_mid, float2* d_out, cudaStream_t st) {
  P2Args a;
  a.y = d_mid;
  a.tw_p2 = ws_ptr<float2>(c, c->lay.tw_p2);
  a.meta = nullptr;
  a.slots = nullptr;
  a.series_rho = nullptr;
  a.series_chi = nullptr;
  a.dense_out = d_out;
  a.p = 1;
  a.n1 = c->n1;
  a.log_n1 = c->log_n - kLogN2;
  a.log_w = 0;
  a.n_windows = 0;
  a.n_rows = c->n1;
  a.thresh = 0.f;
  k_pass2<true, false><<<p2_grid(c, a.n_rows), kP2Warps * 32, kP2Smem, st>>>(a);
  c->launches++;
  return cudaGetLastError();
}

// batch = [bfirst, bfirst + bcount) (pair-aligned: spectra and pass 1 ran for all of it); rows of [first, first + count)
cudaError_t launch_pass2_eff(Ctx* c, int bfirst, int bcount, int first, int count, bool update_slots, float* series_rho,
                             float* series_chi) {
  P2EArgs ea;
  P2Args& a = ea.b;
  a.y = ws_ptr<float2>(c, c->lay.y);
  a.tw_p2 = ws_ptr<float2>(c, c->lay.tw_p2);
  a.meta = ws_ptr<TemplateMeta>(c, c->lay.meta) + bfirst;
  a.slots = update_slots ? ws_ptr<Slot>(c, c->lay.slots) + (size_t)bfirst * c->n_windows : nullptr;
  a.series_rho = series_rho;
  a.series_chi = series_chi;
  a.dense_out = nullptr;
  a.p = c->prm.p;
  a.n1 = c->n1;
  a.log_n1 = c->log_n - kLogN2;
  int lw = 0;
  while ((1 << lw) < c->prm.window) ++lw;
  a.log_w = lw;
  a.n_windows = c->n_windows;
  a.n_rows = count * c->n1;
  a.thresh = (float)c->prm.rho_thresh;
  ea.slot_base = c->h_eff[bfirst];
  ea.log_na = c->log_n - kLogN2 - 5;
  ea.batch = bcount;
  ea.t_begin = first - bfirst;
  const bool single = c->prm.p == 1 || c->prm.chisq_mode == GWMF_CHISQ_ON_DEMAND;   // one effective band per template
  const bool series = series_rho || series_chi;
  const int want = (a.n_rows + kP2EWarps - 1) / kP2EWarps;
  const dim3 grid(want < c->n_sms ? want : c->n_sms);       // persistent: at most one CTA per SM
  if (single && series) k_pass2_eff<true, true><<<grid, kP2EWarps * 32, kP2ESmem, c->stream>>>(ea, c->band_tmap);
  else if (single) k_pass2_eff<false, true><<<grid, kP2EWarps * 32, kP2ESmem, c->stream>>>(ea, c->band_tmap);
  else if (series) k_pass2_eff<true, false><<<grid, kP2EWarps * 32, kP2ESmem, c->stream>>>(ea, c->band_tmap);
  else k_pass2_eff<false, false><<<grid, kP2EWarps * 32, kP2ESmem, c->stream>>>(ea, c->band_tmap);
  c->launches++;
  return cudaGetLastError();
}

}  // namespace gwmf
