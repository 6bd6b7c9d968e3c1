// triggers.cu -- trigger-slot reset and ordered compaction (step a5's output side).
// Events leave the device sorted by (template, window): counts per template, an exclusive scan over
// templates, then each template writes its windows in order.  No atomics, so the order is fixed.
#include "gwmf_internal.cuh"

namespace gwmf {

__global__ void k_reset_slots(Slot* __restrict__ slots, size_t count) {
  size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (i < count) { slots[i].key = 0ull; slots[i].aux = 0ull; }
}

__global__ void k_count(const Slot* __restrict__ slots, int* __restrict__ counts, int n_templates, int n_windows) {
  int t = blockIdx.x * blockDim.x + threadIdx.x;
  if (t >= n_templates) return;
  const Slot* s = slots + (size_t)t * n_windows;
  int c = 0;
  for (int w = 0; w < n_windows; ++w) c += (s[w].key != 0ull);
  counts[t] = c;
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

__global__ void k_emit(const Slot* __restrict__ slots, const long long* __restrict__ offsets,
                       gwmf_trigger* __restrict__ out, long long capacity, int n_templates, int n_windows) {
  int t = blockIdx.x * blockDim.x + threadIdx.x;
  if (t >= n_templates) return;
  const Slot* s = slots + (size_t)t * n_windows;
  long long o = offsets[t];
  for (int w = 0; w < n_windows; ++w) {
    unsigned long long key = s[w].key;
    if (key != 0ull) {
      if (o < capacity) {
        gwmf_trigger g;
        g.template_id = t;
        g.sample = (int32_t)(0xFFFFFFFFu - (unsigned)(key & 0xFFFFFFFFull));
        g.rho = __uint_as_float((unsigned)(key >> 32));
        g.chisq = __uint_as_float((unsigned)(s[w].aux & 0xFFFFFFFFull));
        out[o] = g;
      }
      ++o;
    }
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
  k_count<<<(T + 127) / 128, 128, 0, c->stream>>>(slots, counts, T, c->n_windows);
  k_scan<<<1, 1024, 0, c->stream>>>(counts, offsets, T);
  k_emit<<<(T + 127) / 128, 128, 0, c->stream>>>(slots, offsets, ws_ptr<gwmf_trigger>(c, c->lay.trig_out), cap, T,
                                                 c->n_windows);
  c->launches += 3;
  return cudaGetLastError();
}

}  // namespace gwmf
