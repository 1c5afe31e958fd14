// argus_api.cu — the C ABI of include/argus.h: argument checks, workspace carving, stream/event
// plumbing, launches.  Device memory is allocated in argus_create only (and only when the caller
// passes no workspace); nothing here synchronises the device.
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

// dims the kernels cannot address (ARGUS_ESIZE); cfg_ok(c) holds
static bool cfg_too_large(const argus_config* c) {
  if ((uint64_t)c->n_ranks * c->n_steps >= (1ull << 31)) return true;
  if (argus_record_bytes(c) >= (1ull << 32)) return true;
  if ((uint64_t)c->step_base + c->n_steps > (1ull << 32)) return true;   // step numbers do not wrap (R19)
  if ((uint64_t)c->n_steps * ((uint64_t)c->n_sigs + c->n_phases + 1u) > 0x7FFFFFFFull) return true;   // one CTA per series
  return false;
}

extern "C" size_t argus_record_bytes(const argus_config* c) {
  if (!c) return 0;
  return 64u + 32u * ((size_t)c->n_phases + 1u) + 160u * (size_t)c->n_sigs;
}

extern "C" size_t argus_table_bytes(const argus_config* c) {
  if (!c) return 0;
  return argus_record_bytes(c) * (size_t)c->n_ranks * (size_t)c->n_steps;
}

static size_t up256(size_t v) { return (v + 255u) & ~(size_t)255u; }

void argus_ws_plan(const argus_config* c, int sm_count, int max_smem_optin, argus_ws_layout* L) {
  const size_t RT = (size_t)c->n_ranks * c->n_steps;
  size_t o = 0;
  L->state = o;     o += up256(sizeof(uint32_t) * RT);
  L->counters = o;  o += up256(16 * sizeof(unsigned long long));   // [0..3] events, [4..6] L3 paths, [8] encoder ticket
  L->hist = o;      o += up256(sizeof(uint32_t) * (RT + 1u));
  L->sums = o;      o += up256(sizeof(unsigned long long) * RT * c->n_sigs);
  L->ovf = o;       o += up256((size_t)ARGUS_MAX_SEG_CTAS * ARGUS_OVF_CAP * sizeof(uint4));
  L->diag_todo = o; o += up256((size_t)c->n_steps * ((size_t)c->n_sigs + c->n_phases + 1u));
  L->part = o; L->group = o; L->coarse = o; L->part_ctas = 0; L->part_smem = false;
  L->part_two_level = false; L->part_shift = 0;
  if (c->max_ungrouped_events) {
    size_t small = 0;
    L->part_two_level = (size_t)max_smem_optin >= 100u * 1024u && argus_partition2_plan(c, &L->part_shift, &small);
    if (L->part_two_level) {
      o += up256(small);
      L->coarse = o;
      o += up256((size_t)c->max_ungrouped_events * 16u);
    } else {
      argus_partition_plan(c, sm_count, max_smem_optin, &L->part_ctas, &L->part_smem);
      if (L->part_smem) o += up256(sizeof(uint32_t) * (size_t)L->part_ctas * (RT + 1u));
    }
    L->group = o;
    o += up256((size_t)c->max_ungrouped_events * sizeof(argus_event));
  }
  L->spill = o;
  if (c->max_spill_events) o += up256((size_t)c->max_spill_events * 8u);
  L->total = o;
}

static cudaError_t device_shape(int device, int* sm_count, int* max_smem_optin) {
  cudaError_t e = cudaDeviceGetAttribute(sm_count, cudaDevAttrMultiProcessorCount, device);
  if (e == cudaSuccess) e = cudaDeviceGetAttribute(max_smem_optin, cudaDevAttrMaxSharedMemoryPerBlockOptin, device);
  return e;
}

extern "C" size_t argus_workspace_bytes(const argus_config* cfg) {
  if (!cfg_ok(cfg) || cfg_too_large(cfg)) return 0;
  int sms = 0, smem = 0;
  if (device_shape(cfg->device, &sms, &smem) != cudaSuccess) { (void)cudaGetLastError(); return 0; }
  argus_ws_layout L;
  argus_ws_plan(cfg, sms, smem, &L);
  return L.total;
}

extern "C" int argus_create(const argus_config* cfg, void* d_workspace, size_t workspace_bytes, argus_ctx** out) {
  if (!out) return ARGUS_EINVAL;
  *out = nullptr;
  if (!cfg_ok(cfg)) return ARGUS_EINVAL;
  if (cfg_too_large(cfg)) return ARGUS_ESIZE;
  if (d_workspace && ((uintptr_t)d_workspace & 255u)) return ARGUS_EINVAL;
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
  int code = ARGUS_OK;
  cudaError_t e = cudaSetDevice(cfg->device);
  if (e == cudaSuccess) e = device_shape(cfg->device, &ctx->sm_count, &ctx->max_smem_optin);
  if (e == cudaSuccess) {
    argus_ws_plan(cfg, ctx->sm_count, ctx->max_smem_optin, &ctx->ws);
    if (d_workspace) {
      if (workspace_bytes < ctx->ws.total) code = ARGUS_EINVAL;
      ctx->d_ws = static_cast<uint8_t*>(d_workspace);
    } else {
      void* p = nullptr;
      e = cudaMalloc(&p, ctx->ws.total);     // the library's only device allocation
      ctx->d_ws = static_cast<uint8_t*>(p);
      ctx->ws_owned = e == cudaSuccess;
    }
  }
  if (e == cudaSuccess && code == ARGUS_OK) {
    const argus_ws_layout& L = ctx->ws;
    ctx->d_state = reinterpret_cast<uint32_t*>(ctx->d_ws + L.state);
    ctx->d_counters = reinterpret_cast<unsigned long long*>(ctx->d_ws + L.counters);
    ctx->d_hist = reinterpret_cast<uint32_t*>(ctx->d_ws + L.hist);
    D.sums = reinterpret_cast<unsigned long long*>(ctx->d_ws + L.sums);
    ctx->d_ovf = reinterpret_cast<uint4*>(ctx->d_ws + L.ovf);
    ctx->d_diag_todo = ctx->d_ws + L.diag_todo;
    if (cfg->max_spill_events) ctx->d_spill = ctx->d_ws + L.spill;
    if (cfg->max_ungrouped_events) {
      ctx->d_part = (L.part_smem || L.part_two_level) ? reinterpret_cast<uint32_t*>(ctx->d_ws + L.part) : nullptr;
      ctx->d_coarse = L.part_two_level ? ctx->d_ws + L.coarse : nullptr;
      ctx->d_group = reinterpret_cast<argus_event*>(ctx->d_ws + L.group);
    }
    cudaDriverEntryPointQueryResult q;
    void* fn = nullptr;
    if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &fn, cudaEnableDefault, &q) == cudaSuccess &&
        q == cudaDriverEntryPointSuccess)
      ctx->fn_tmap_encode = fn;
    (void)cudaGetLastError();
    e = cudaEventCreateWithFlags(&ctx->ingest_event, cudaEventDisableTiming);
    if (e == cudaSuccess) e = cudaEventCreateWithFlags(&ctx->order_event, cudaEventDisableTiming);
    if (e == cudaSuccess) e = cudaStreamCreateWithFlags(&ctx->copy_stream, cudaStreamNonBlocking);
    if (e == cudaSuccess) e = argus_configure_kernels(ctx);   // opt-in shared-memory sizes, once
  }
  if (e != cudaSuccess || code != ARGUS_OK) {
    if (e != cudaSuccess) {
      code = (e == cudaErrorMemoryAllocation) ? ARGUS_ENOMEM : ARGUS_ECUDA;
      (void)cudaGetLastError();
    }
    argus_destroy(ctx);
    return code;
  }
  *out = ctx;
  return ARGUS_OK;
}

extern "C" int argus_destroy(argus_ctx* ctx) {
  if (!ctx) return ARGUS_EINVAL;
  cudaSetDevice(ctx->cfg.device);
  if (ctx->ws_owned && ctx->d_ws) cudaFree(ctx->d_ws);
  if (ctx->ingest_event) cudaEventDestroy(ctx->ingest_event);
  if (ctx->order_event) cudaEventDestroy(ctx->order_event);
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

// argus_stats synchronises every stream the ctx was given; remember the distinct ones
static int note_stream(argus_ctx* ctx, cudaStream_t s) {
  for (uint32_t i = 0; i < ctx->n_streams; ++i)
    if (ctx->streams[i] == s) return ARGUS_OK;
  if (ctx->n_streams == 8u) {
    CU(ctx, cudaStreamSynchronize(ctx->streams[0]));
    memmove(&ctx->streams[0], &ctx->streams[1], 7 * sizeof(cudaStream_t));
    ctx->n_streams = 7u;
  }
  ctx->streams[ctx->n_streams++] = s;
  return ARGUS_OK;
}

extern "C" int argus_reset(argus_ctx* ctx, void* d_records, void* stream) {
  if (!ctx || !d_records || !aligned16(d_records)) return ARGUS_EINVAL;
  cudaStream_t s = (cudaStream_t)stream;
  CU(ctx, cudaSetDevice(ctx->cfg.device));
  int rc = note_stream(ctx, s);
  if (rc != ARGUS_OK) return rc;
  // state words and counters are neighbours in the workspace: one memset
  CU(ctx, cudaMemsetAsync(ctx->d_state, 0, ctx->ws.hist - ctx->ws.state, s));
  ctx->n_memsets += 1;
  ctx->d_records = d_records;
  ctx->finalized = false;
  return ARGUS_OK;
}

extern "C" int argus_ingest(argus_ctx* ctx, const argus_event* h_src, uint64_t n, argus_event* d_dst,
                            void* copy_stream) {
  if (!ctx) return ARGUS_EINVAL;
  if (n == 0) return ARGUS_OK;
  if (!h_src || !d_dst || !aligned16(d_dst)) return ARGUS_EINVAL;
  cudaStream_t cs = (cudaStream_t)copy_stream;
  CU(ctx, cudaSetDevice(ctx->cfg.device));
  int rc = note_stream(ctx, cs);
  if (rc != ARGUS_OK) return rc;
  CU(ctx, cudaMemcpyAsync(d_dst, h_src, n * sizeof(argus_event), cudaMemcpyHostToDevice, cs));
  CU(ctx, cudaEventRecord(ctx->ingest_event, cs));
  ctx->ingest_pending = true;
  return ARGUS_OK;
}

// Path choice: grouped input (ARGUS_FLAG_SORTED) -> segmented kernel; ungrouped input -> group the
// events by (rank, step) first, then the segmented kernel; the global-table kernel is what is left
// when the table does not fit the segmented kernel or the call exceeds the grouping area.
static int aggregate_impl(argus_ctx* ctx, const argus_event* d_events, uint64_t n, void* d_records,
                          cudaStream_t s) {
  int path = ctx->tune_path;
  if (path == 0) path = (ctx->cfg.flags & ARGUS_FLAG_SORTED) ? 1 : 3;
  if ((path == 1 || path == 3) && !argus_seg_supported(ctx)) path = 2;
  if (path == 3 && n > ctx->cfg.max_ungrouped_events) path = 2;
  if (path == 3) {
    CU(ctx, argus_launch_partition(ctx, d_events, n, s));
    d_events = ctx->d_group;
    path = 1;
  }
  if (path == 1) CU(ctx, argus_launch_aggregate_seg(ctx, d_events, n, d_records, s));
  else CU(ctx, argus_launch_aggregate_global(ctx, d_events, n, d_records, s));
  return ARGUS_OK;
}

// the next kernel on `s` must see the bytes of the last argus_ingest
static int wait_ingest(argus_ctx* ctx, cudaStream_t s) {
  if (ctx->ingest_pending) {
    CU(ctx, cudaStreamWaitEvent(s, ctx->ingest_event, 0));
    ctx->ingest_pending = false;
  }
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
  int rc = note_stream(ctx, s);
  if (rc == ARGUS_OK) rc = wait_ingest(ctx, s);
  if (rc != ARGUS_OK || n == 0) return rc;
  ctx->finalized = false;
  return aggregate_impl(ctx, d_events, n, d_records, s);
}

static int ensure_slot_events(argus_ctx* ctx, uint32_t ring_slots) {
  if (ctx->n_slot_events >= ring_slots) return ARGUS_OK;
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
  return ARGUS_OK;
}

extern "C" int argus_aggregate_host(argus_ctx* ctx, const argus_event* h_events, uint64_t n,
                                    uint64_t chunk_events, argus_event* d_ring, uint32_t ring_slots,
                                    void* d_records, void* stream) {
  if (!ctx || !d_records) return ARGUS_EINVAL;
  if (d_records != ctx->d_records) return ARGUS_ESTATE;
  cudaStream_t s = (cudaStream_t)stream;
  CU(ctx, cudaSetDevice(ctx->cfg.device));
  int rc = note_stream(ctx, s);
  if (rc == ARGUS_OK) rc = wait_ingest(ctx, s);    // an argus_ingest the caller queued before us stays ordered
  if (rc != ARGUS_OK || n == 0) return rc;
  if (!h_events || !d_ring || !aligned16(d_ring) || ring_slots == 0 || ring_slots > 64u || chunk_events == 0)
    return ARGUS_EINVAL;
  if (chunk_events >= (1ull << 32)) return ARGUS_ESIZE;
  rc = ensure_slot_events(ctx, ring_slots);
  if (rc != ARGUS_OK) return rc;
  ctx->finalized = false;
  // the copy stream must not run ahead of work already queued on `stream` that may still read the
  // ring (an earlier call): order it after the compute stream's current tail
  CU(ctx, cudaEventRecord(ctx->order_event, s));
  CU(ctx, cudaStreamWaitEvent(ctx->copy_stream, ctx->order_event, 0));
  const uint64_t n_chunks = (n + chunk_events - 1) / chunk_events;
  for (uint64_t c = 0; c < n_chunks; ++c) {
    const uint32_t slot = (uint32_t)(c % ring_slots);
    const uint64_t cnt = (c + 1 == n_chunks) ? n - c * chunk_events : chunk_events;
    argus_event* dst = d_ring + (size_t)slot * chunk_events;
    // slot reuse: the copy of chunk c waits for the aggregation of chunk c - ring_slots
    if (c >= ring_slots) CU(ctx, cudaStreamWaitEvent(ctx->copy_stream, ctx->slot_free[slot], 0));
    CU(ctx, cudaMemcpyAsync(dst, h_events + c * chunk_events, cnt * sizeof(argus_event),
                            cudaMemcpyHostToDevice, ctx->copy_stream));
    CU(ctx, cudaEventRecord(ctx->slot_full[slot], ctx->copy_stream));
    CU(ctx, cudaStreamWaitEvent(s, ctx->slot_full[slot], 0));
    rc = aggregate_impl(ctx, dst, cnt, d_records, s);
    if (rc != ARGUS_OK) return rc;
    CU(ctx, cudaEventRecord(ctx->slot_free[slot], s));
  }
  return ARGUS_OK;
}

extern "C" int argus_phase_times(argus_ctx* ctx, void* d_records, argus_span* d_spans_out, void* stream) {
  if (!ctx || !d_records) return ARGUS_EINVAL;
  if (d_records != ctx->d_records) return ARGUS_ESTATE;
  if (d_spans_out && !aligned16(d_spans_out)) return ARGUS_EINVAL;
  cudaStream_t s = (cudaStream_t)stream;
  CU(ctx, cudaSetDevice(ctx->cfg.device));
  int rc = note_stream(ctx, s);
  if (rc != ARGUS_OK) return rc;
  CU(ctx, argus_launch_finalize(ctx, d_records, d_spans_out, s));
  ctx->finalized = true;
  return ARGUS_OK;
}

extern "C" int argus_diagnose(argus_ctx* ctx, const void* d_records, const argus_diag_out* outs, void* stream) {
  if (!ctx || !d_records || !outs || !aligned16(d_records)) return ARGUS_EINVAL;
  if ((outs->sig_stats && !aligned16(outs->sig_stats)) || (outs->span_stats && !aligned16(outs->span_stats)))
    return ARGUS_EINVAL;
  if (((uintptr_t)outs->rank_score & 3u) || ((uintptr_t)outs->step_anomalous & 3u)) return ARGUS_EINVAL;
  // our own table must be finalised (span_ns, headers, identities of untouched records); a foreign
  // finalised table (e.g. one read back from storage) is gathered from its records
  const bool own = d_records == ctx->d_records;
  if (own && !ctx->finalized) return ARGUS_ESTATE;
  cudaStream_t s = (cudaStream_t)stream;
  CU(ctx, cudaSetDevice(ctx->cfg.device));
  int rc = note_stream(ctx, s);
  if (rc != ARGUS_OK) return rc;
  CU(ctx, argus_launch_diagnose(ctx, d_records, outs, /*use_sums=*/own, s));
  return ARGUS_OK;
}

extern "C" int argus_forget(argus_ctx* ctx) {
  if (!ctx) return ARGUS_EINVAL;
  ctx->d_records = nullptr;      // no address compares equal to it any more: every table is foreign
  ctx->finalized = false;
  return ARGUS_OK;
}

static bool aligned8(const void* p) { return ((uintptr_t)p & 7u) == 0; }

extern "C" int argus_pack_planes(argus_ctx* ctx, const void* d_records, uint32_t sig_lo, uint32_t sig_hi,
                                 uint64_t* d_sig_plane, uint64_t* d_span_plane, uint32_t rank_stride,
                                 uint32_t rank_offset, void* stream) {
  if (!ctx || !d_records) return ARGUS_EINVAL;
  if (d_records != ctx->d_records || !ctx->finalized) return ARGUS_ESTATE;   // the sum plane mirrors OUR table
  if (sig_lo > sig_hi || sig_hi > ctx->dims.S) return ARGUS_EINVAL;
  if (!aligned8(d_sig_plane) || !aligned8(d_span_plane)) return ARGUS_EINVAL;
  if ((uint64_t)rank_offset + ctx->dims.R > rank_stride) return ARGUS_EINVAL;
  cudaStream_t s = (cudaStream_t)stream;
  CU(ctx, cudaSetDevice(ctx->cfg.device));
  int rc = note_stream(ctx, s);
  if (rc != ARGUS_OK) return rc;
  CU(ctx, argus_launch_pack_planes(ctx, d_records, sig_lo, sig_hi, d_sig_plane, d_span_plane, rank_stride,
                                   rank_offset, s));
  return ARGUS_OK;
}

extern "C" int argus_diagnose_planes(argus_ctx* ctx, const argus_planes* pl, const argus_diag_out* outs,
                                     void* stream) {
  if (!ctx || !pl || !outs) return ARGUS_EINVAL;
  if (pl->n_ranks == 0 || pl->n_ranks > ARGUS_MAX_RANKS || pl->rank_stride < pl->n_ranks) return ARGUS_EINVAL;
  if (pl->n_sigs > ctx->dims.S || (pl->n_sigs != 0) != (pl->sig_sums != nullptr)) return ARGUS_EINVAL;
  if (!aligned8(pl->sig_sums) || !aligned8(pl->span_ns)) return ARGUS_EINVAL;
  if ((outs->sig_stats && !aligned16(outs->sig_stats)) || (outs->span_stats && !aligned16(outs->span_stats)))
    return ARGUS_EINVAL;
  if (((uintptr_t)outs->rank_score & 3u) || ((uintptr_t)outs->step_anomalous & 3u)) return ARGUS_EINVAL;
  cudaStream_t s = (cudaStream_t)stream;
  CU(ctx, cudaSetDevice(ctx->cfg.device));
  int rc = note_stream(ctx, s);
  if (rc != ARGUS_OK) return rc;
  CU(ctx, argus_launch_diagnose_planes(ctx, pl, outs, s));
  return ARGUS_OK;
}

// ---- the paper-literal float algorithms (paper_literal.cu) ------------------------------------------------
static bool kde_params_ok(const argus_kde_params* p) {
  return p && (p->per_octave == 1u || p->per_octave == 8u) && p->n_bins >= 2u && p->n_bins <= 256u &&
         p->max_clusters >= 1u && p->max_clusters <= 16u && p->min_frac >= 0.0;
}

#define ARGUS_ENTER(ctx, stream)                       \
  cudaStream_t s = (cudaStream_t)(stream);             \
  CU(ctx, cudaSetDevice((ctx)->cfg.device));           \
  {                                                    \
    int rc__ = note_stream(ctx, s);                    \
    if (rc__ != ARGUS_OK) return rc__;                 \
  }

extern "C" int argus_fine_hist(argus_ctx* ctx, const argus_event* d_events, uint64_t n, uint32_t* d_hist, void* stream) {
  if (!ctx || !d_hist || ((uintptr_t)d_hist & 3u)) return ARGUS_EINVAL;
  if (n != 0 && (!d_events || !aligned16(d_events))) return ARGUS_EINVAL;
  ARGUS_ENTER(ctx, stream);
  CU(ctx, argus_launch_fine_hist(ctx, d_events, n, d_hist, s));
  return ARGUS_OK;
}

extern "C" int argus_kde_clusters(argus_ctx* ctx, const uint32_t* d_hist, uint64_t n_cells, const argus_kde_params* p,
                                  argus_cluster* d_clusters, uint8_t* d_n_clusters, double* d_density, void* stream) {
  if (!ctx || !kde_params_ok(p) || !d_hist || !d_clusters || !d_n_clusters) return ARGUS_EINVAL;
  if (((uintptr_t)d_hist & 3u) || !aligned8(d_clusters) || !aligned8(d_density)) return ARGUS_EINVAL;
  if ((n_cells + 7) / 8 > 0x7FFFFFFFull) return ARGUS_ESIZE;
  ARGUS_ENTER(ctx, stream);
  CU(ctx, argus_launch_kde_hist(ctx, d_hist, n_cells, p, d_clusters, d_n_clusters, d_density, s));
  return ARGUS_OK;
}

extern "C" int argus_kde_clusters_records(argus_ctx* ctx, const void* d_records, const argus_kde_params* p,
                                          argus_cluster* d_clusters, uint8_t* d_n_clusters, void* stream) {
  if (!ctx || !kde_params_ok(p) || p->n_bins != 32u || p->per_octave != 1u) return ARGUS_EINVAL;
  if (!d_records || !d_clusters || !d_n_clusters || !aligned8(d_clusters)) return ARGUS_EINVAL;
  if (d_records == ctx->d_records && !ctx->finalized) return ARGUS_ESTATE;
  if (((uint64_t)ctx->dims.R * ctx->dims.T * ctx->dims.S + 7) / 8 > 0x7FFFFFFFull) return ARGUS_ESIZE;
  ARGUS_ENTER(ctx, stream);
  CU(ctx, argus_launch_kde_records(ctx, d_records, p, d_clusters, d_n_clusters, s));
  return ARGUS_OK;
}

extern "C" size_t argus_sparse_bound(const argus_config* c) {
  if (!cfg_ok(c)) return 0;
  return (size_t)c->n_ranks * c->n_steps * (72u + 32u * (size_t)c->n_phases + 168u * (size_t)c->n_sigs);
}

extern "C" size_t argus_triple_bound(const argus_config* c, uint32_t max_clusters) {
  if (!cfg_ok(c) || max_clusters == 0) return 0;
  return (size_t)c->n_ranks * c->n_steps * (72u + 32u * (size_t)c->n_phases + (8u + 8u * (size_t)max_clusters) * c->n_sigs);
}

extern "C" int argus_sparse_encode(argus_ctx* ctx, const void* d_records, uint8_t* d_out, uint64_t out_capacity,
                                   uint64_t* d_offsets, void* stream) {
  if (!ctx || !d_records || !d_out || !d_offsets || !aligned8(d_out) || !aligned8(d_offsets)) return ARGUS_EINVAL;
  if (d_records == ctx->d_records && !ctx->finalized) return ARGUS_ESTATE;
  ARGUS_ENTER(ctx, stream);
  CU(ctx, argus_launch_sparse_encode(ctx, d_records, d_out, out_capacity, d_offsets, s));
  return ARGUS_OK;
}

extern "C" int argus_triple_encode(argus_ctx* ctx, const void* d_records, const argus_cluster* d_clusters,
                                   const uint8_t* d_n_clusters, uint32_t max_clusters, uint8_t* d_out,
                                   uint64_t out_capacity, uint64_t* d_offsets, void* stream) {
  if (!ctx || !d_records || !d_clusters || !d_n_clusters || !d_out || !d_offsets || max_clusters == 0) return ARGUS_EINVAL;
  if (!aligned8(d_clusters) || !aligned8(d_out) || !aligned8(d_offsets)) return ARGUS_EINVAL;
  if (d_records == ctx->d_records && !ctx->finalized) return ARGUS_ESTATE;
  ARGUS_ENTER(ctx, stream);
  CU(ctx, argus_launch_triple_encode(ctx, d_records, d_clusters, d_n_clusters, max_clusters, d_out, out_capacity, d_offsets, s));
  return ARGUS_OK;
}

extern "C" int argus_clusters_to_l3(argus_ctx* ctx, const argus_cluster* d_clusters, uint32_t max_clusters,
                                    uint32_t per_octave, uint32_t* d_count, double* d_p50, double* d_p99, void* stream) {
  if (!ctx || !d_clusters || !d_count || !d_p50 || !d_p99 || max_clusters == 0 || per_octave == 0) return ARGUS_EINVAL;
  if (!aligned8(d_clusters) || !aligned8(d_p50) || !aligned8(d_p99) || ((uintptr_t)d_count & 3u)) return ARGUS_EINVAL;
  ARGUS_ENTER(ctx, stream);
  CU(ctx, argus_launch_clusters_to_l3(ctx, d_clusters, max_clusters, per_octave, d_count, d_p50, d_p99, s));
  return ARGUS_OK;
}

extern "C" int argus_l3_detect(argus_ctx* ctx, const argus_l3_in* in, const argus_l3_params* p, double* d_score,
                               argus_l3_stat* d_stat, uint8_t* d_flags, void* stream) {
  if (!ctx || !in || !p || !d_score || !d_stat || !d_flags) return ARGUS_EINVAL;
  if (in->n_keys != 0 && (!in->count || !in->p50 || !in->p99)) return ARGUS_EINVAL;
  if (in->n_ranks == 0 || in->max_clusters == 0 || p->n_grid < 2u) return ARGUS_EINVAL;
  if (in->n_ranks > 4096u || argus_l3_smem_bytes(in->n_ranks) > (size_t)ctx->max_smem_optin) return ARGUS_ESIZE;
  if (!aligned8(d_score) || !aligned8(d_stat) || !aligned8(in->p50) || !aligned8(in->p99)) return ARGUS_EINVAL;
  ARGUS_ENTER(ctx, stream);
  CU(ctx, argus_launch_l3(ctx, in, p, d_score, d_stat, d_flags, s));
  return ARGUS_OK;
}

extern "C" int argus_l2_groups(argus_ctx* ctx, const void* d_records, const uint8_t* d_route, uint32_t n_dims,
                               const uint32_t* d_group_id, double z_threshold, argus_l2_group* d_groups, double* d_z, uint8_t* d_flags,
                               double* d_xbar, void* stream) {
  if (!ctx || !d_records || !d_route || !d_group_id || !d_groups || !d_z || !d_flags || !d_xbar) return ARGUS_EINVAL;
  if (n_dims == 0 || n_dims > 256u) return ARGUS_EINVAL;          // a route entry is one byte
  if (!aligned8(d_groups) || !aligned8(d_z) || !aligned8(d_xbar) || ((uintptr_t)d_group_id & 3u)) return ARGUS_EINVAL;
  if (d_records == ctx->d_records && !ctx->finalized) return ARGUS_ESTATE;
  ARGUS_ENTER(ctx, stream);
  CU(ctx, argus_launch_l2(ctx, d_records, d_route, n_dims, d_group_id, z_threshold, d_groups, d_z, d_flags, d_xbar, s));
  return ARGUS_OK;
}

extern "C" int argus_l1_detect(argus_ctx* ctx, const void* d_base, uint64_t series_stride, uint64_t step_stride,
                               uint32_t n_series, uint32_t n_steps, const argus_l1_params* p, argus_l1_out* d_out,
                               void* stream) {
  if (!ctx || !p || !d_out || !aligned8(d_out)) return ARGUS_EINVAL;
  if (n_series != 0 && n_steps != 0 && (!d_base || !aligned8(d_base) || (series_stride & 7u) || (step_stride & 7u)))
    return ARGUS_EINVAL;
  if (p->window < 2u || p->min_seg < 2u) return ARGUS_EINVAL;
  if (n_steps > 2048u) return ARGUS_ESIZE;
  ARGUS_ENTER(ctx, stream);
  CU(ctx, argus_launch_l1(ctx, d_base, series_stride, step_stride, n_series, n_steps, p, d_out, s));
  return ARGUS_OK;
}

extern "C" int argus_stats(argus_ctx* ctx, uint64_t* n_valid, uint64_t* n_invalid) {
  if (!ctx) return ARGUS_EINVAL;
  CU(ctx, cudaSetDevice(ctx->cfg.device));
  CU(ctx, cudaStreamSynchronize(ctx->copy_stream));
  for (uint32_t i = 0; i < ctx->n_streams; ++i) CU(ctx, cudaStreamSynchronize(ctx->streams[i]));
  unsigned long long h[2] = {0, 0};
  CU(ctx, cudaMemcpy(h, ctx->d_counters, sizeof h, cudaMemcpyDeviceToHost));
  h[0] -= h[1];  // kernels count events seen and events rejected
  if (n_valid) *n_valid = h[0];
  if (n_invalid) *n_invalid = h[1];
  return ARGUS_OK;
}

extern "C" int argus_refused_count(argus_ctx* ctx, uint64_t* n_requeued, uint64_t* n_overflow) {
  if (!ctx) return ARGUS_EINVAL;
  int rc = argus_stats(ctx, nullptr, nullptr);      // synchronises the streams
  if (rc != ARGUS_OK) return rc;
  unsigned long long h[2] = {0, 0};
  CU(ctx, cudaMemcpy(h, ctx->d_counters + 2, sizeof h, cudaMemcpyDeviceToHost));
  if (n_overflow) *n_overflow = h[0];
  if (n_requeued) *n_requeued = h[1];
  return ARGUS_OK;
}

extern "C" int argus_l3_path_count(argus_ctx* ctx, uint64_t* n_class, uint64_t* n_general, uint64_t* n_empty) {
  if (!ctx) return ARGUS_EINVAL;
  int rc = argus_stats(ctx, nullptr, nullptr);      // synchronises the streams
  if (rc != ARGUS_OK) return rc;
  unsigned long long h[3] = {0, 0, 0};
  CU(ctx, cudaMemcpy(h, ctx->d_counters + 4, sizeof h, cudaMemcpyDeviceToHost));
  if (n_class) *n_class = h[0];
  if (n_general) *n_general = h[1];
  if (n_empty) *n_empty = h[2];
  return ARGUS_OK;
}

extern "C" int argus_launch_count(const argus_ctx* ctx, uint64_t* kernels, uint64_t* memsets) {
  if (!ctx) return ARGUS_EINVAL;
  if (kernels) *kernels = ctx->n_kernels;
  if (memsets) *memsets = ctx->n_memsets;
  return ARGUS_OK;
}

extern "C" int argus_tune(argus_ctx* ctx, int which, int64_t value) {
  if (!ctx) return ARGUS_EINVAL;
  switch (which) {
    case ARGUS_TUNE_GRID_CTAS:
      if (value < 0 || value > (int64_t)ARGUS_MAX_SEG_CTAS) return ARGUS_EINVAL;
      ctx->tune_grid = (int)value;
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
extern "C" const char* argus_version(void) { return "argus-b200 0.2.0 (sm_100a)"; }
