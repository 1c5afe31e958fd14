// aggregate_global.cu — global-table aggregation (BASELINE.json configs[3]: "records shuffled
// uniformly across rank-steps, so aggregation cannot rely on contiguous segments and must use
// global hashed/dense-table accumulation"), plus the identity materialisation it needs.
//
// Every record is first made LIVE (identity bytes of R7 written, state word set), then each event
// is folded straight into its dense cell with L2 reductions (RED.ADD/MIN/MAX).  The table
// (1.3 GB at config 3) is far larger than L2, so this path is bound by random 32-byte sector
// read-modify-writes in HBM, not by the 32 B/event stream; DESIGN.md §6.2.
#include "argus_internal.cuh"

namespace {

// Identity-fill every record whose state is LAZY and mark it LIVE.  One CTA walks records.
__global__ void materialise_kernel(uint8_t* records, uint32_t* state, argus_dims D, uint32_t n_rec) {
  const uint32_t n_chunks = 2u * (D.P + 1u) + 10u * D.S;
  for (uint32_t rec = blockIdx.x; rec < n_rec; rec += gridDim.x) {
    if (state[rec] != ARGUS_ST_LAZY) continue;   // uniform per CTA; nobody else runs on this stream
    uint4* dst = reinterpret_cast<uint4*>(records + (size_t)rec * D.rec_bytes + D.span_off);
    for (uint32_t ch = threadIdx.x; ch < n_chunks; ch += blockDim.x) dst[ch] = argus_identity_chunk(D, ch);
    argus_zero_sums_row(D, rec, threadIdx.x, blockDim.x);
    __syncthreads();
    if (threadIdx.x == 0) state[rec] = ARGUS_ST_LIVE;
  }
}

__global__ void __launch_bounds__(256)
aggregate_global_kernel(const uint4* __restrict__ ev, uint64_t n, uint8_t* records,
                        unsigned long long* counters, argus_dims D) {
  uint32_t n_valid = 0, n_invalid = 0;   // counters[0] counts events SEEN, counters[1] rejected
  const uint64_t stride = (uint64_t)gridDim.x * blockDim.x;
  const int lane = threadIdx.x & 31;
  // lane pairs fetch the two 16-byte halves of an event as ONE coalesced 512-byte warp access per
  // 16 events; a shuffle hands the second half to the lane that processes the event
  for (uint64_t base = ((uint64_t)blockIdx.x * blockDim.x + threadIdx.x - lane); base < n; base += stride) {
    // this warp covers events [base, base+32): two coalesced loads of 32 uint4 each
    uint4 a = make_uint4(0, 0, 0, 0), b = make_uint4(0, 0, 0, 0);
    const uint64_t q0 = 2 * base + lane, q1 = 2 * base + 32 + lane;
    if (q0 < 2 * n) a = __ldcs(ev + q0);
    if (q1 < 2 * n) b = __ldcs(ev + q1);
    // lane 2k holds lo(ev k) in a and lo(ev 16+k) in b; lane 2k+1 holds hi(ev k), hi(ev 16+k).
    // even lanes process ev k, odd lanes process ev 16+k.
    const bool odd = lane & 1;
    uint4 give = odd ? a : b;        // what the neighbour needs
    uint4 got;
    got.x = __shfl_xor_sync(0xFFFFFFFFu, give.x, 1);
    got.y = __shfl_xor_sync(0xFFFFFFFFu, give.y, 1);
    got.z = __shfl_xor_sync(0xFFFFFFFFu, give.z, 1);
    got.w = __shfl_xor_sync(0xFFFFFFFFu, give.w, 1);
    const uint4 lo = odd ? got : a;
    const uint4 hi = odd ? b : got;
    const uint64_t idx = base + (odd ? 16 + (lane >> 1) : (lane >> 1));
    if (idx < n) {
      ++n_valid;
      const uint32_t phase = lo.w >> 16;
      const long long start = (long long)(((unsigned long long)hi.y << 32) | hi.x);
      const long long end = (long long)(((unsigned long long)hi.w << 32) | hi.z);
      uint32_t key;
      if (argus_event_key(D, lo.x, lo.y, lo.z, phase, start, end, key)) {
        argus_global_accumulate(records + (size_t)key * D.rec_bytes, key, D, lo.z, phase, start, end);
      } else {
        ++n_invalid;
      }
    }
  }
  n_valid = __reduce_add_sync(0xFFFFFFFFu, n_valid);
  n_invalid = __reduce_add_sync(0xFFFFFFFFu, n_invalid);
  if (lane == 0) {
    if (n_valid) atomicAdd(&counters[0], (unsigned long long)n_valid);
    if (n_invalid) atomicAdd(&counters[1], (unsigned long long)n_invalid);
  }
}

}  // namespace

cudaError_t argus_launch_materialise_all(argus_ctx* ctx, void* d_records, cudaStream_t s) {
  const uint32_t n_rec = ctx->dims.R * ctx->dims.T;
  uint32_t grid = n_rec < (uint32_t)ctx->sm_count * 8u ? n_rec : (uint32_t)ctx->sm_count * 8u;
  materialise_kernel<<<grid, 256, 0, s>>>(static_cast<uint8_t*>(d_records), ctx->d_state, ctx->dims, n_rec);
  ctx->n_kernels += 1;
  return cudaGetLastError();
}

cudaError_t argus_launch_aggregate_global(argus_ctx* ctx, const argus_event* ev, uint64_t n,
                                          void* d_records, cudaStream_t s) {
  if (n == 0) return cudaSuccess;
  cudaError_t e = argus_launch_materialise_all(ctx, d_records, s);
  if (e != cudaSuccess) return e;
  uint64_t blocks = (n + 255) / 256;
  const uint64_t cap = (uint64_t)ctx->sm_count * 32;
  if (blocks > cap) blocks = cap;
  aggregate_global_kernel<<<(unsigned)blocks, 256, 0, s>>>(reinterpret_cast<const uint4*>(ev), n,
                                                           static_cast<uint8_t*>(d_records),
                                                           ctx->d_counters, ctx->dims);
  ctx->n_kernels += 1;
  return cudaGetLastError();
}
