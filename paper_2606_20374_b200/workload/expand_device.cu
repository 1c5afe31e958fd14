/* expand_device.cu — device build of the workload expander (see expand_core.h): one thread per
 * rank, same integer code as the host build, so the bytes are identical.  Used by bench.py and the
 * full-size tests to fill HBM with tens of GB of events without a host round trip.
 * Input generator only: none of the method's arithmetic lives here. */
#include "expand_core.h"
#include <cuda_runtime.h>

__global__ void wl_expand_kernel(wl_desc d, uint32_t rank_lo, uint32_t rank_hi, wl_event* out) {
  uint32_t r = rank_lo + blockIdx.x * blockDim.x + threadIdx.x;
  if (r >= rank_hi) return;
  const uint64_t per_rank = (uint64_t)d.n_steps * d.n_events;
  if (d.shuffle) wl_expand_rank(&d, r, out, 0);
  else wl_expand_rank(&d, r, out + (uint64_t)(r - rank_lo) * per_rank, (uint64_t)r * per_rank);
}

/* d: [host] struct whose table pointers are [device] pointers.  out: [device].  Asynchronous on
 * stream.  Returns 0 or the cudaError_t of the launch. */
extern "C" int wl_expand_device(const wl_desc* d, uint32_t rank_lo, uint32_t rank_hi, wl_event* out,
                                void* stream) {
  if (!d || !out || rank_lo > rank_hi || rank_hi > d->n_ranks || d->n_streams > WL_MAX_STREAMS ||
      d->n_streams == 0)
    return -1;
  uint32_t n = rank_hi - rank_lo;
  if (n == 0) return 0;
  const int threads = 32;
  wl_expand_kernel<<<(n + threads - 1) / threads, threads, 0, (cudaStream_t)stream>>>(
      *d, rank_lo, rank_hi, out);
  return (int)cudaGetLastError();
}
