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
