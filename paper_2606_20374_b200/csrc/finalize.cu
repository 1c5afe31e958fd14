// finalize.cu — argus_phase_times: the summary encoder's last step (NS (5), R17).  Never re-reads
// events.  One CTA per record: materialise the identities of an untouched record (lazy reset),
// set span_ns of every phase span, derive the whole-iteration span (index P) as the hull of the
// phase spans (NS: "Iteration time is max(end) minus min(start) over a rank-step, and phase time
// uses the same rule within each phase"), write the 64-byte header.
#include "argus_internal.cuh"

namespace {

__global__ void __launch_bounds__(256)
finalize_kernel(uint8_t* records, uint32_t* state, argus_span* spans_out, argus_dims D, uint32_t n_rec) {
  __shared__ long long s_mn[ARGUS_MAX_PHASES], s_mx[ARGUS_MAX_PHASES];
  __shared__ unsigned long long s_n[ARGUS_MAX_PHASES];
  const uint32_t n_chunks = 2u * (D.P + 1u) + 10u * D.S;
  for (uint32_t rec = blockIdx.x; rec < n_rec; rec += gridDim.x) {
    uint8_t* base = records + (size_t)rec * D.rec_bytes;
    if (state[rec] == ARGUS_ST_LAZY) {
      uint4* dst = reinterpret_cast<uint4*>(base + D.span_off);
      for (uint32_t ch = threadIdx.x; ch < n_chunks; ch += blockDim.x) dst[ch] = argus_identity_chunk(D, ch);
      argus_zero_sums_row(D, rec, threadIdx.x, blockDim.x);
      __syncthreads();
      if (threadIdx.x == 0) state[rec] = ARGUS_ST_LIVE;
    }
    __syncthreads();
    argus_span* sp = reinterpret_cast<argus_span*>(base + D.span_off);
    for (uint32_t k = threadIdx.x; k < D.P; k += blockDim.x) {
      argus_span v = sp[k];
      v.span_ns = v.n_events ? (uint64_t)(v.max_end_ns - v.min_start_ns) : 0ull;
      sp[k].span_ns = v.span_ns;
      s_mn[k] = v.min_start_ns; s_mx[k] = v.max_end_ns; s_n[k] = v.n_events;
      if (spans_out) spans_out[(size_t)rec * (D.P + 1) + k] = v;
    }
    __syncthreads();
    if (threadIdx.x == 0) {
      argus_span w;
      w.min_start_ns = INT64_MAX; w.max_end_ns = INT64_MIN; w.n_events = 0;
      for (uint32_t k = 0; k < D.P; ++k) {
        w.min_start_ns = s_mn[k] < w.min_start_ns ? s_mn[k] : w.min_start_ns;
        w.max_end_ns = s_mx[k] > w.max_end_ns ? s_mx[k] : w.max_end_ns;
        w.n_events += s_n[k];
      }
      w.span_ns = w.n_events ? (uint64_t)(w.max_end_ns - w.min_start_ns) : 0ull;
      sp[D.P] = w;
      if (spans_out) spans_out[(size_t)rec * (D.P + 1) + D.P] = w;
      argus_record_header h;
      h.magic = ARGUS_RECORD_MAGIC; h.version = ARGUS_RECORD_VERSION; h.n_phases = (uint16_t)D.P;
      h.n_sigs = D.S; h.rank = rec / D.T; h.step = D.step_base + rec % D.T; h.reserved0 = 0;
      h.n_events = w.n_events; h.min_start_ns = w.min_start_ns; h.max_end_ns = w.max_end_ns;
      h.iter_ns = w.span_ns; h.reserved1 = 0;
      *reinterpret_cast<argus_record_header*>(base) = h;
    }
    __syncthreads();
  }
}

}  // namespace

cudaError_t argus_launch_finalize(argus_ctx* ctx, void* d_records, argus_span* d_spans_out,
                                  cudaStream_t s) {
  const uint32_t n_rec = ctx->dims.R * ctx->dims.T;
  uint32_t grid = n_rec < (uint32_t)ctx->sm_count * 8u ? n_rec : (uint32_t)ctx->sm_count * 8u;
  finalize_kernel<<<grid, 256, 0, s>>>(static_cast<uint8_t*>(d_records), ctx->d_state, d_spans_out,
                                       ctx->dims, n_rec);
  ctx->n_kernels += 1;
  return cudaGetLastError();
}
