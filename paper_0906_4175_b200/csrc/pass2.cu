// pass2.cu -- second pass of the band inverse FFTs fused with the statistics and the trigger maxima
// (second half of step a3, steps a4 and a5).
//
// One warp owns one output residue j1 and walks over the p bands.  For each band the contiguous
// 1024-point row Y_l[j1][0..1023] (8 KB) is brought into the warp's shared-memory buffer by one TMA bulk
// copy (cp.async.bulk + mbarrier), issued one band ahead so that HBM latency hides behind the previous
// band's arithmetic; the warp transforms it in registers (32 x 32, one transpose through the same
// buffer, re-read with row stride 33) and accumulates, per output sample it owns,
//     z   = sum_l z_l            (Sigma_l z_l = z: no separate full-band transform)
//     q   = sum_l |z_l|^2
// so that rho^2 = |z|^2 / sigma^2 (Eq. 3) and chi^2 = (p/sigma^2)(q - |z|^2/p), which is Eq. 5
// by the identity sum_l |z_l - z/p|^2 = sum_l |z_l|^2 - |z|^2/p.  The band series never
// reach HBM.  Samples with rho > threshold race for their (template, window) slot with a 128-bit
// compare-and-swap on (rho, -index | chi^2): the result is the maximum, lowest index on ties,
// whatever the order of arrival.
#include "fft_reg.cuh"
#include "gwmf_internal.cuh"

namespace gwmf {

struct P2Args {
  const float2* y;            // [batch][p][n1][1024]
  const float2* tw_p2;        // [32][32] e^{2 pi i jm c/1024}
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

constexpr int kRowBytes = kN2 * (int)sizeof(float2);      // 8 KB
constexpr int kBufElems = 32 * 33;                        // row buffer, also the stride-33 transpose tile

// Shared memory: [tw 32x32][warp 0: buf0, buf1][warp 1: ...]...[mbarriers 2 per warp].
// A warp's current input buffer doubles as its transpose tile (row stride 33 -> conflict-free both ways).
template <bool STORE>
__global__ void __launch_bounds__(kP2Warps * 32) k_pass2(P2Args a) {
  extern __shared__ __align__(128) float2 smem2[];
  float2* tw_s = smem2;                                   // [32][32]
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  float2* bufs = smem2 + 1024 + warp * (2 * kBufElems);   // two row buffers
  unsigned long long* bars = reinterpret_cast<unsigned long long*>(smem2 + 1024 + kP2Warps * 2 * kBufElems) + 2 * warp;

  const int j1 = blockIdx.x * kP2Warps + warp;
  const int tb = blockIdx.y;
  const int p = a.p;
  const float2* row0 = a.y + ((size_t)(tb * p) * a.n1 + j1) * kN2;
  const size_t band_stride = (size_t)a.n1 * kN2;

  unsigned long long policy;
  asm volatile("createpolicy.fractional.L2::evict_first.b64 %0, 1.0;" : "=l"(policy));
  if (lane == 0) {
    mbar_init(&bars[0], 1);
    mbar_init(&bars[1], 1);
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
    mbar_expect_tx(&bars[0], kRowBytes);
    bulk_load_row(bufs, row0, kRowBytes, &bars[0], policy);
  }
  for (int i = threadIdx.x; i < 1024; i += blockDim.x) tw_s[i] = a.tw_p2[i];
  __syncthreads();

  float2 az[32];
  float aq[32];
#pragma unroll
  for (int i = 0; i < 32; ++i) { az[i] = make_float2(0.f, 0.f); aq[i] = 0.f; }

#pragma unroll 1
  for (int l = 0; l < p; ++l) {
    float2* cur = bufs + (l & 1) * kBufElems;
    if (l + 1 < p && lane == 0) {
      // the other buffer was last touched (generic proxy) in iteration l-1: order that before the async write
      asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
      mbar_expect_tx(&bars[(l + 1) & 1], kRowBytes);
      bulk_load_row(bufs + ((l + 1) & 1) * kBufElems, row0 + (size_t)(l + 1) * band_stride, kRowBytes, &bars[(l + 1) & 1], policy);
    }
    mbar_wait(&bars[l & 1], (l >> 1) & 1);
    float2 x[32];
#pragma unroll
    for (int m = 0; m < 32; ++m) x[brev<32>(m)] = cur[32 * m + lane];     // k2 = 32 m + lane
    __syncwarp();
    fft_dit<32>(x);                                                       // over m -> jm
#pragma unroll
    for (int jm = 0; jm < 32; ++jm)
      cur[jm * 33 + lane] = cmul(x[jm], tw_s[jm * 32 + lane]);   // times e^{2 pi i jm c/1024}
    __syncwarp();
#pragma unroll
    for (int cc = 0; cc < 32; ++cc) x[brev<32>(cc)] = cur[lane * 33 + cc];   // now lane = jm, index = c
    __syncwarp();
    fft_dit<32>(x);                                                       // over c -> jc; j2 = lane + 32 jc
    if constexpr (STORE) {
#pragma unroll
      for (int jc = 0; jc < 32; ++jc)
        a.dense_out[(size_t)j1 + ((size_t)(lane + 32 * jc) << a.log_n1)] = x[jc];
    } else {
#pragma unroll
      for (int jc = 0; jc < 32; ++jc) {
        const float2 z = x[jc];
        az[jc] = cadd(az[jc], z);
        aq[jc] = fmaf(z.x, z.x, fmaf(z.y, z.y, aq[jc]));
      }
    }
  }

  if constexpr (!STORE) {
    const TemplateMeta* m = a.meta + tb;
    const float scale = m->scale_rho2;
    const float fp = (float)p, inv_p = 1.0f / (float)p;
    const float thr2 = a.thresh * a.thresh;
#pragma unroll
    for (int jc = 0; jc < 32; ++jc) {
      const float z2 = fmaf(az[jc].x, az[jc].x, az[jc].y * az[jc].y);
      const float rho2 = z2 * scale;                                        // Eq. 3 squared
      const float chi = fmaxf(aq[jc] - z2 * inv_p, 0.f) * (fp * scale);     // Eq. 5
      const unsigned j = (unsigned)j1 + ((unsigned)(lane + 32 * jc) << a.log_n1);
      if (a.series_rho) a.series_rho[j] = sqrtf(rho2);
      if (a.series_chi) a.series_chi[j] = chi;
      if (a.slots && rho2 > thr2 * 0.999f) {
        const float rho = sqrtf(rho2);
        if (rho > a.thresh) {
          Slot* s = a.slots + (size_t)tb * a.n_windows + (j >> a.log_w);
          slot_max(s, ((unsigned long long)__float_as_uint(rho) << 32) | (unsigned long long)(0xFFFFFFFFu - j),
                   (unsigned long long)__float_as_uint(chi));
        }
      }
    }
  }
}

constexpr size_t kP2Smem = (1024 + kP2Warps * 2 * kBufElems) * sizeof(float2) + kP2Warps * 2 * sizeof(unsigned long long);

static cudaError_t p2_configure() {
  static bool done = false;
  if (done) return cudaSuccess;
  cudaError_t e = cudaFuncSetAttribute(k_pass2<false>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)kP2Smem);
  if (e == cudaSuccess) e = cudaFuncSetAttribute(k_pass2<true>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)kP2Smem);
  done = (e == cudaSuccess);
  return e;
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
  a.thresh = (float)c->prm.rho_thresh;
  dim3 grid(c->n1 / kP2Warps, count);
  cudaError_t e = p2_configure();
  if (e != cudaSuccess) return e;
  k_pass2<false><<<grid, kP2Warps * 32, kP2Smem, c->stream>>>(a);
  c->launches++;
  return cudaGetLastError();
}

cudaError_t launch_pass2_dense(Ctx* c, const float2* d_mid, float2* d_out) {
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
  a.thresh = 0.f;
  dim3 grid(c->n1 / kP2Warps, 1);
  cudaError_t e = p2_configure();
  if (e != cudaSuccess) return e;
  k_pass2<true><<<grid, kP2Warps * 32, kP2Smem, c->stream>>>(a);
  c->launches++;
  return cudaGetLastError();
}

}  // namespace gwmf
