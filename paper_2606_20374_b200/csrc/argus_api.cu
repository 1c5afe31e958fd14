// argus_api.cu — the C ABI of include/argus.h: argument checks, stream/event plumbing, launches.
#include <new>
#include <string.h>

#include "argus_internal.cuh"

#define CU(ctx, call)                                   \
  do {                                                  \
    cudaError_t e__ = (call);                           \
    if (e__ != cudaSuccess) {                           \
      (ctx)->last_cuda_error = (int)e__;                \
      return ARGUS_ECUDA;                               \
    }                                                   \
  } while (0)

static bool cfg_ok(const argus_config* c) {
  if (!c) return false;
  if (c->n_ranks == 0 || c->n_ranks > ARGUS_MAX_RANKS) return false;
  if (c->n_steps == 0 || c->n_sigs == 0) return false;
  if (c->n_phases == 0 || c->n_phases > ARGUS_MAX_PHASES) return false;
  return true;
}

extern "C" size_t argus_record_bytes(const argus_config* c) {
  if (!c) return 0;
  return 64u + 32u * ((size_t)c->n_phases + 1u) + 160u * (size_t)c->n_sigs;
}

extern "C" size_t argus_table_bytes(const argus_config* c) {
  if (!c) return 0;
  return argus_record_bytes(c) * (size_t)c->n_ranks * (size_t)c->n_steps;
}

extern "C" int argus_create(const argus_config* cfg, argus_ctx** out) {
  if (!out) return ARGUS_EINVAL;
  *out = nullptr;
  if (!cfg_ok(cfg)) return ARGUS_EINVAL;
  if ((uint64_t)cfg->n_ranks * cfg->n_steps >= (1ull << 31)) return ARGUS_ESIZE;
  if (argus_record_bytes(cfg) >= (1ull << 32)) return ARGUS_ESIZE;
  argus_ctx* ctx = new (std::nothrow) argus_ctx();
  if (!ctx) return ARGUS_ENOMEM;
  memset(ctx, 0, sizeof *ctx);
  ctx->cfg = *cfg;
  argus_dims& D = ctx->dims;
  D.R = cfg->n_ranks; D.T = cfg->n_steps; D.S = cfg->n_sigs; D.P = cfg->n_phases;
  D.step_base = cfg->step_base;
  D.rec_bytes = (uint32_t)argus_record_bytes(cfg);
  D.span_off = 64u;
  D.cell_off = 64u + 32u * (D.P + 1u);
  cudaError_t e = cudaSetDevice(cfg->device);
  cudaDeviceProp prop;
  if (e == cudaSuccess) e = cudaGetDeviceProperties(&prop, cfg->device);
  if (e == cudaSuccess) {
    ctx->sm_count = prop.multiProcessorCount;
    ctx->max_smem_optin = (int)prop.sharedMemPerBlockOptin;
    e = cudaMalloc(&ctx->d_state, sizeof(uint32_t) * (size_t)D.R * D.T);
  }
  if (e == cudaSuccess) {
    cudaDriverEntryPointQueryResult q;
    void* fn = nullptr;
    if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &fn, cudaEnableDefault, &q) == cudaSuccess &&
        q == cudaDriverEntryPointSuccess)
      ctx->fn_tmap_encode = fn;
    (void)cudaGetLastError();
  }
  if (e == cudaSuccess) {
    // the sum plane (8 bytes per cell, 5 % of the table) is an accelerator of argus_diagnose only:
    // without it the gather falls back to the records
    if (cudaMalloc(&D.sums, sizeof(unsigned long long) * (size_t)D.R * D.T * D.S) != cudaSuccess) {
      D.sums = nullptr;
      (void)cudaGetLastError();
    }
  }
  if (e == cudaSuccess) e = cudaMalloc(&ctx->d_counters, 2 * sizeof(unsigned long long));
  if (e == cudaSuccess) e = cudaMalloc(&ctx->d_hist, sizeof(uint32_t) * ((size_t)D.R * D.T + 1u));
  if (e == cudaSuccess) e = cudaEventCreateWithFlags(&ctx->ingest_event, cudaEventDisableTiming);
  if (e == cudaSuccess) e = cudaStreamCreateWithFlags(&ctx->copy_stream, cudaStreamNonBlocking);
  if (e != cudaSuccess) {
    int code = (e == cudaErrorMemoryAllocation) ? ARGUS_ENOMEM : ARGUS_ECUDA;
    argus_destroy(ctx);
    return code;
  }
  *out = ctx;
  return ARGUS_OK;
}

extern "C" int argus_destroy(argus_ctx* ctx) {
  if (!ctx) return ARGUS_EINVAL;
  cudaSetDevice(ctx->cfg.device);
  if (ctx->d_state) cudaFree(ctx->d_state);
  if (ctx->d_counters) cudaFree(ctx->d_counters);
  if (ctx->dims.sums) cudaFree(ctx->dims.sums);
  if (ctx->d_hist) cudaFree(ctx->d_hist);
  if (ctx->d_group) cudaFree(ctx->d_group);
  if (ctx->d_ovf) cudaFree(ctx->d_ovf);
  if (ctx->d_diag_todo) cudaFree(ctx->d_diag_todo);
  if (ctx->d_part) cudaFree(ctx->d_part);
  if (ctx->ingest_event) cudaEventDestroy(ctx->ingest_event);
  for (uint32_t i = 0; i < ctx->n_slot_events; ++i) {
    cudaEventDestroy(ctx->slot_free[i]);
    cudaEventDestroy(ctx->slot_full[i]);
  }
  delete[] ctx->slot_free;
  delete[] ctx->slot_full;
  if (ctx->copy_stream) cudaStreamDestroy(ctx->copy_stream);
  delete ctx;
  return ARGUS_OK;
}

static bool aligned16(const void* p) { return ((uintptr_t)p & 15u) == 0; }

extern "C" int argus_reset(argus_ctx* ctx, void* d_records, void* stream) {
  if (!ctx || !d_records || !aligned16(d_records)) return ARGUS_EINVAL;
  cudaStream_t s = (cudaStream_t)stream;
  CU(ctx, cudaSetDevice(ctx->cfg.device));
  CU(ctx, cudaMemsetAsync(ctx->d_state, 0, sizeof(uint32_t) * (size_t)ctx->dims.R * ctx->dims.T, s));
  CU(ctx, cudaMemsetAsync(ctx->d_counters, 0, 2 * sizeof(unsigned long long), s));
  ctx->d_records = d_records;
  ctx->finalized = false;
  ctx->last_stream = s;
  return ARGUS_OK;
}

extern "C" int argus_ingest(argus_ctx* ctx, const argus_event* h_src, uint64_t n, argus_event* d_dst,
                            void* copy_stream) {
  if (!ctx) return ARGUS_EINVAL;
  if (n == 0) return ARGUS_OK;
  if (!h_src || !d_dst || !aligned16(d_dst)) return ARGUS_EINVAL;
  cudaStream_t cs = (cudaStream_t)copy_stream;
  CU(ctx, cudaSetDevice(ctx->cfg.device));
  CU(ctx, cudaMemcpyAsync(d_dst, h_src, n * sizeof(argus_event), cudaMemcpyHostToDevice, cs));
  CU(ctx, cudaEventRecord(ctx->ingest_event, cs));
  ctx->ingest_pending = true;
  return ARGUS_OK;
}

// Path choice: grouped input (ARGUS_FLAG_SORTED) -> segmented kernel; ungrouped input -> group the
// events by (rank, step) first, then the segmented kernel; the global-table kernel is what is left
// when the table does not fit the segmented kernel or the grouping workspace cannot be allocated.
static int aggregate_impl(argus_ctx* ctx, const argus_event* d_events, uint64_t n, void* d_records,
                          cudaStream_t s) {
  int path = ctx->tune_path;
  if (path == 0) path = (ctx->cfg.flags & ARGUS_FLAG_SORTED) ? 1 : 3;
  if ((path == 1 || path == 3) && !argus_seg_supported(ctx)) path = 2;
  if (path == 3) {
    cudaError_t e = argus_launch_partition(ctx, d_events, n, s);
    if (e == cudaErrorMemoryAllocation) path = 2;
    else {
      CU(ctx, e);
      d_events = ctx->d_group;
      path = 1;
    }
  }
  if (path == 1) CU(ctx, argus_launch_aggregate_seg(ctx, d_events, n, d_records, s));
  else CU(ctx, argus_launch_aggregate_global(ctx, d_events, n, d_records, s));
  return ARGUS_OK;
}

extern "C" int argus_aggregate(argus_ctx* ctx, const argus_event* d_events, uint64_t n,
                               void* d_records, void* stream) {
  if (!ctx || !d_records) return ARGUS_EINVAL;
  if (d_records != ctx->d_records) return ARGUS_ESTATE;
  if (n >= (1ull << 32)) return ARGUS_ESIZE;
  if (n != 0 && (!d_events || !aligned16(d_events))) return ARGUS_EINVAL;
  cudaStream_t s = (cudaStream_t)stream;
  CU(ctx, cudaSetDevice(ctx->cfg.device));
  if (ctx->ingest_pending) {
    CU(ctx, cudaStreamWaitEvent(s, ctx->ingest_event, 0));
    ctx->ingest_pending = false;
  }
  ctx->last_stream = s;
  if (n == 0) return ARGUS_OK;
  return aggregate_impl(ctx, d_events, n, d_records, s);
}

extern "C" int argus_aggregate_host(argus_ctx* ctx, const argus_event* h_events, uint64_t n,
                                    uint64_t chunk_events, argus_event* d_ring, uint32_t ring_slots,
                                    void* d_records, void* stream) {
  if (!ctx || !d_records) return ARGUS_EINVAL;
  if (d_records != ctx->d_records) return ARGUS_ESTATE;
  if (n == 0) return ARGUS_OK;
  if (!h_events || !d_ring || !aligned16(d_ring) || ring_slots == 0 || chunk_events == 0)
    return ARGUS_EINVAL;
  if (chunk_events >= (1ull << 32)) return ARGUS_ESIZE;
  cudaStream_t s = (cudaStream_t)stream;
  CU(ctx, cudaSetDevice(ctx->cfg.device));
  if (ctx->n_slot_events < ring_slots) {
    cudaEvent_t* f = new (std::nothrow) cudaEvent_t[ring_slots];
    cudaEvent_t* u = new (std::nothrow) cudaEvent_t[ring_slots];
    if (!f || !u) { delete[] f; delete[] u; return ARGUS_ENOMEM; }
    for (uint32_t i = 0; i < ctx->n_slot_events; ++i) { f[i] = ctx->slot_free[i]; u[i] = ctx->slot_full[i]; }
    uint32_t made = ctx->n_slot_events;
    for (; made < ring_slots; ++made) {
      if (cudaEventCreateWithFlags(&f[made], cudaEventDisableTiming) != cudaSuccess) break;
      if (cudaEventCreateWithFlags(&u[made], cudaEventDisableTiming) != cudaSuccess) {
        cudaEventDestroy(f[made]);
        break;
      }
    }
    delete[] ctx->slot_free;
    delete[] ctx->slot_full;
    ctx->slot_free = f; ctx->slot_full = u; ctx->n_slot_events = made;
    if (made < ring_slots) { ctx->last_cuda_error = (int)cudaGetLastError(); return ARGUS_ECUDA; }
  }
  // the copy stream must not run ahead of work already queued on `stream` that may still read the
  // ring (an earlier call): order it after the compute stream's current tail
  CU(ctx, cudaEventRecord(ctx->ingest_event, s));
  CU(ctx, cudaStreamWaitEvent(ctx->copy_stream, ctx->ingest_event, 0));
  const uint64_t n_chunks = (n + chunk_events - 1) / chunk_events;
  for (uint64_t c = 0; c < n_chunks; ++c) {
    const uint32_t slot = (uint32_t)(c % ring_slots);
    const uint64_t cnt = (c + 1 == n_chunks) ? n - c * chunk_events : chunk_events;
    argus_event* dst = d_ring + (size_t)slot * chunk_events;
    if (c >= ring_slots) CU(ctx, cudaStreamWaitEvent(ctx->copy_stream, ctx->slot_free[slot], 0));
    CU(ctx, cudaMemcpyAsync(dst, h_events + c * chunk_events, cnt * sizeof(argus_event),
                            cudaMemcpyHostToDevice, ctx->copy_stream));
    CU(ctx, cudaEventRecord(ctx->slot_full[slot], ctx->copy_stream));
    CU(ctx, cudaStreamWaitEvent(s, ctx->slot_full[slot], 0));
    int rc = aggregate_impl(ctx, dst, cnt, d_records, s);
    if (rc != ARGUS_OK) return rc;
    CU(ctx, cudaEventRecord(ctx->slot_free[slot], s));
  }
  ctx->last_stream = s;
  return ARGUS_OK;
}

extern "C" int argus_phase_times(argus_ctx* ctx, void* d_records, argus_span* d_spans_out, void* stream) {
  if (!ctx || !d_records) return ARGUS_EINVAL;
  if (d_records != ctx->d_records) return ARGUS_ESTATE;
  if (d_spans_out && !aligned16(d_spans_out)) return ARGUS_EINVAL;
  cudaStream_t s = (cudaStream_t)stream;
  CU(ctx, cudaSetDevice(ctx->cfg.device));
  ctx->last_stream = s;
  CU(ctx, argus_launch_finalize(ctx, d_records, d_spans_out, s));
  ctx->finalized = true;
  return ARGUS_OK;
}

extern "C" int argus_diagnose(argus_ctx* ctx, const void* d_records, const argus_diag_out* outs, void* stream) {
  if (!ctx || !d_records || !outs || !aligned16(d_records)) return ARGUS_EINVAL;
  if ((outs->sig_stats && !aligned16(outs->sig_stats)) || (outs->span_stats && !aligned16(outs->span_stats)))
    return ARGUS_EINVAL;
  cudaStream_t s = (cudaStream_t)stream;
  CU(ctx, cudaSetDevice(ctx->cfg.device));
  ctx->last_stream = s;
  // the sum plane mirrors the table given to argus_reset, finalised by argus_phase_times
  const bool use_sums = ctx->dims.sums != nullptr && d_records == ctx->d_records && ctx->finalized;
  CU(ctx, argus_launch_diagnose(ctx, d_records, outs, use_sums, s));
  return ARGUS_OK;
}

extern "C" int argus_stats(argus_ctx* ctx, uint64_t* n_valid, uint64_t* n_invalid) {
  if (!ctx) return ARGUS_EINVAL;
  CU(ctx, cudaSetDevice(ctx->cfg.device));
  CU(ctx, cudaStreamSynchronize(ctx->copy_stream));
  CU(ctx, cudaStreamSynchronize(ctx->last_stream));
  unsigned long long h[2] = {0, 0};
  CU(ctx, cudaMemcpy(h, ctx->d_counters, sizeof h, cudaMemcpyDeviceToHost));
  h[0] -= h[1];  // kernels count events seen and events rejected
  if (n_valid) *n_valid = h[0];
  if (n_invalid) *n_invalid = h[1];
  return ARGUS_OK;
}

extern "C" int argus_tune(argus_ctx* ctx, int which, int64_t value) {
  if (!ctx) return ARGUS_EINVAL;
  switch (which) {
    case ARGUS_TUNE_GRID_CTAS:
      if (value < 0 || value > 65535) return ARGUS_EINVAL;
      ctx->tune_grid = (int)value;
      return ARGUS_OK;
    case ARGUS_TUNE_SEG_VARIANT:
      ctx->tune_variant = (int)value;
      return ARGUS_OK;
    case ARGUS_TUNE_FORCE_PATH:
      if (value < 0 || value > 3) return ARGUS_EINVAL;
      ctx->tune_path = (int)value;
      return ARGUS_OK;
    default:
      return ARGUS_EINVAL;
  }
}

extern "C" const char* argus_strerror(int code) {
  switch (code) {
    case ARGUS_OK: return "ok";
    case ARGUS_EINVAL: return "invalid argument";
    case ARGUS_ECUDA: return "CUDA error (see argus_last_cuda_error)";
    case ARGUS_ESIZE: return "size out of range";
    case ARGUS_ESTATE: return "call order violated";
    case ARGUS_ENOMEM: return "out of memory";
    default: return "unknown error";
  }
}

extern "C" int argus_last_cuda_error(const argus_ctx* ctx) { return ctx ? ctx->last_cuda_error : 0; }
extern "C" const char* argus_version(void) { return "argus-b200 0.1.0 (sm_100a)"; }
