// argus_internal.cuh — shared declarations of libargus.so (CUDA side only; never seen by the oracle).
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

#include "argus.h"

// ---- per-record state words (ctx workspace, one u32 per (rank, step)) -------------------------
// 0: identity, bytes of the record not written yet (lazy argus_reset)
// 2: one CTA holds the claim and is writing the record with plain stores
// 1: materialised — every further contribution merges with atomics
#define ARGUS_ST_LAZY 0u
#define ARGUS_ST_BUSY 2u
#define ARGUS_ST_LIVE 1u

struct argus_dims {
  uint32_t R, T, S, P, step_base;
  uint32_t rec_bytes;   // 64 + 32*(P+1) + 160*S
  uint32_t span_off;    // 64
  uint32_t cell_off;    // 64 + 32*(P+1)
  // Sum plane (workspace; null in kernels that must not touch it): sums[(rank*T + t)*S + sig] mirrors cell.sum_ns of the table
  // given to argus_reset, sig-contiguous, so that the cross-rank gather of argus_diagnose reads whole
  // sectors of neighbouring sigs instead of one 32-byte sector per 160-byte cell.  Every kernel that
  // writes a cell's sum (flush, merge, global path, identity fill) keeps it in step.
  unsigned long long* sums;
};

// Areas of the device workspace (argus_workspace_bytes): byte offsets from its base, each 256-byte
// aligned; computed by one function so that argus_workspace_bytes and argus_create cannot disagree.
#define ARGUS_MAX_SEG_CTAS 1024u      // CTAs of one segmented launch (bounds the overflow-list area)
#define ARGUS_OVF_CAP 4096u           // entries (16 B) of one CTA's overflow list
struct argus_ws_layout {
  size_t state, counters, hist, sums, ovf, diag_todo, part, group, spill, total;
  size_t coarse;                      // two-level grouping: the packed events grouped by coarse bin (16 B per event)
  uint32_t part_ctas;                 // CTAs of the grouping pass (0: no grouping area)
  bool part_smem;                     // its key histograms fit shared memory
  bool part_two_level;                // two-level grouping (partition.cu) instead of the single scatter
  uint32_t part_shift;                // keys per coarse bin = 2^part_shift
};
void argus_ws_plan(const argus_config* cfg, int sm_count, int max_smem_optin, argus_ws_layout* out);

struct argus_ctx {
  argus_config cfg;
  argus_dims dims;
  int sm_count;
  int max_smem_optin;
  argus_ws_layout ws;
  uint8_t* d_ws;              // the workspace (caller's, or ours when ws_owned)
  bool ws_owned;
  uint32_t* d_state;          // [R*T]
  unsigned long long* d_counters;  // [4] events seen, rejected, taken by the overflow list / L2 atomics, re-queued
  uint32_t* d_hist;           // [R*T + 1] group sizes / cursors of the grouping pass
  argus_event* d_group;       // grouping area [cfg.max_ungrouped_events] (null when 0)
  void* fn_tmap_encode;       // cuTensorMapEncodeTiled, resolved through the runtime (no libcuda link)
  uint32_t* d_part;           // per-CTA key histograms of the grouping pass [part_ctas][R*T + 1], or the small
                              // state of the two-level pass
  uint8_t* d_coarse;          // two-level grouping: coarse area [cfg.max_ungrouped_events] x 16 B
  uint8_t* d_diag_todo;       // argus_diagnose: one byte per series, set by the 32-bit pass for the 64-bit pass
  uint8_t* d_spill;           // spill regions of the segmented kernel: {sig, duration} of re-queued events, 8 B x cfg.max_spill_events (null when 0)
  uint4* d_ovf;               // per-CTA overflow lists of the segmented kernel [ARGUS_MAX_SEG_CTAS][ARGUS_OVF_CAP]
  void* d_records;            // table given to the last argus_reset
  cudaEvent_t ingest_event;   // recorded after every argus_ingest copy
  cudaEvent_t order_event;    // argus_aggregate_host: orders the copy stream after the compute stream's tail
  bool ingest_pending;
  bool finalized;             // argus_phase_times ran since the last argus_reset / argus_aggregate
  cudaStream_t copy_stream;   // internal, for argus_aggregate_host
  cudaEvent_t* slot_free;     // ring-slot reuse events (argus_aggregate_host)
  cudaEvent_t* slot_full;
  uint32_t n_slot_events;
  cudaStream_t streams[8];    // distinct streams seen since argus_create (argus_stats synchronises them)
  uint32_t n_streams;
  int last_cuda_error;
  int tune_grid;
  int tune_path;
  uint64_t n_kernels, n_memsets;   // launches since argus_create (argus_launch_count)
};

// kernels' host-side launchers (each returns cudaError_t of the launch)
cudaError_t argus_launch_aggregate_seg(argus_ctx* ctx, const argus_event* ev, uint64_t n,
                                       void* d_records, cudaStream_t s);
cudaError_t argus_launch_aggregate_global(argus_ctx* ctx, const argus_event* ev, uint64_t n,
                                          void* d_records, cudaStream_t s);
cudaError_t argus_launch_partition(argus_ctx* ctx, const argus_event* ev, uint64_t n, cudaStream_t s);
cudaError_t argus_launch_materialise_all(argus_ctx* ctx, void* d_records, cudaStream_t s);
cudaError_t argus_launch_finalize(argus_ctx* ctx, void* d_records, argus_span* d_spans_out,
                                  cudaStream_t s);
cudaError_t argus_launch_diagnose(argus_ctx* ctx, const void* d_records, const argus_diag_out* o,
                                  bool use_sums, cudaStream_t s);
cudaError_t argus_launch_diagnose_planes(argus_ctx* ctx, const argus_planes* pl, const argus_diag_out* o,
                                         cudaStream_t s);
cudaError_t argus_launch_pack_planes(argus_ctx* ctx, const void* d_records, uint32_t s0, uint32_t s1,
                                     uint64_t* dst_sig, uint64_t* dst_span, uint32_t stride, uint32_t off,
                                     cudaStream_t s);
cudaError_t argus_launch_fine_hist(argus_ctx* ctx, const argus_event* ev, uint64_t n, uint32_t* d_hist, cudaStream_t s);
cudaError_t argus_launch_kde_hist(argus_ctx* ctx, const uint32_t* d_hist, uint64_t n_cells, const argus_kde_params* P,
                                  argus_cluster* d_clusters, uint8_t* d_n, double* d_density, cudaStream_t s);
cudaError_t argus_launch_kde_records(argus_ctx* ctx, const void* d_records, const argus_kde_params* P,
                                     argus_cluster* d_clusters, uint8_t* d_n, cudaStream_t s);
cudaError_t argus_launch_clusters_to_l3(argus_ctx* ctx, const argus_cluster* d_clusters, uint32_t mc, uint32_t per_octave,
                                        uint32_t* d_count, double* d_p50, double* d_p99, cudaStream_t s);
cudaError_t argus_launch_sparse_encode(argus_ctx* ctx, const void* d_records, uint8_t* d_out, uint64_t capacity,
                                       uint64_t* d_offsets, cudaStream_t s);
cudaError_t argus_launch_triple_encode(argus_ctx* ctx, const void* d_records, const argus_cluster* d_clusters,
                                       const uint8_t* d_n_clusters, uint32_t mc, uint8_t* d_out, uint64_t capacity,
                                       uint64_t* d_offsets, cudaStream_t s);
size_t argus_l3_smem_bytes(uint32_t R);
cudaError_t argus_launch_l3(argus_ctx* ctx, const argus_l3_in* in, const argus_l3_params* P, double* d_score,
                            argus_l3_stat* d_stat, uint8_t* d_flags, cudaStream_t s);
cudaError_t argus_launch_l2(argus_ctx* ctx, const void* d_records, const uint8_t* d_route, uint32_t n_dims,
                            const uint32_t* d_group_id, double z_thr, argus_l2_group* d_groups, double* d_z, uint8_t* d_flags, double* d_xbar,
                            cudaStream_t s);
cudaError_t argus_launch_l1(argus_ctx* ctx, const void* d_base, uint64_t sstride, uint64_t tstride, uint32_t n_series,
                            uint32_t T, const argus_l1_params* P, argus_l1_out* d_out, cudaStream_t s);
bool argus_seg_supported(const argus_ctx* ctx);
void argus_partition_plan(const argus_config* cfg, int sm_count, int max_smem_optin, uint32_t* n_cta,
                          bool* smem);
bool argus_partition2_plan(const argus_config* cfg, uint32_t* shift, size_t* small_bytes);
// opt-in shared-memory sizes of the kernels this ctx will launch (argus_create, once)
cudaError_t argus_configure_seg(argus_ctx* ctx);
cudaError_t argus_configure_partition(argus_ctx* ctx);
cudaError_t argus_configure_compact(argus_ctx* ctx);
cudaError_t argus_configure_paper_literal(argus_ctx* ctx);
inline cudaError_t argus_configure_kernels(argus_ctx* ctx) {
  cudaError_t e = argus_configure_seg(ctx);
  if (e == cudaSuccess) e = argus_configure_partition(ctx);
  if (e == cudaSuccess) e = argus_configure_compact(ctx);
  return e == cudaSuccess ? argus_configure_paper_literal(ctx) : e;
}
// Let `kernel` ask for all the dynamic shared memory the device can give it (what is left beside its static
// arrays).  The attribute is per function and process-wide: setting it ONCE, in argus_create, to a value that
// does not depend on the call means contexts on other threads can only ever write the same number.
template <typename K>
inline cudaError_t argus_optin_all_smem(K kernel, int max_smem_optin) {
  cudaFuncAttributes a;
  cudaError_t e = cudaFuncGetAttributes(&a, kernel);
  if (e != cudaSuccess) return e;
  return cudaFuncSetAttribute(kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, max_smem_optin - (int)a.sharedSizeBytes);
}

// ---- device helpers shared by the kernels ------------------------------------------------------
#ifdef __CUDACC__

// R4: bucket(d) = d==0 ? 0 : min(31, floor(log2 d)), with count-leading-zeros.
__device__ __forceinline__ uint32_t argus_bucket64(uint64_t d) {
  uint32_t b = 63u - (uint32_t)__clzll((long long)(d | 1ull));
  return b > 31u ? 31u : b;
}

// Event validity (R2, R3) and the dense record index key = rank*T + (step - step_base).
__device__ __forceinline__ bool argus_event_key(const argus_dims& D, uint32_t rank, uint32_t step,
                                                uint32_t sig, uint32_t phase, int64_t start,
                                                int64_t end, uint32_t& key) {
  uint32_t t = step - D.step_base;  // wraps to >= T when step < step_base (T*R < 2^31)
  bool ok = (rank < D.R) & (t < D.T) & (sig < D.S) & (phase < D.P) & (start >= 0) & (end >= start);
  key = rank * D.T + t;
  return ok;
}

// One event straight into a LIVE record with L2 atomics (global-table path, and the overflow path
// of the segmented kernel).  min/max and span bounds are tested first: after the first few events
// of a cell they rarely improve, so most events cost 3 reductions (count, sum, hist) + 1 (span n).
__device__ __forceinline__ void argus_global_accumulate(uint8_t* rec, uint32_t key, const argus_dims& D,
                                                        uint32_t sig, uint32_t phase, int64_t start,
                                                        int64_t end) {
  uint64_t d = (uint64_t)(end - start);
  argus_cell* c = reinterpret_cast<argus_cell*>(rec + D.cell_off) + sig;
  atomicAdd(reinterpret_cast<unsigned long long*>(&c->count), 1ull);
  atomicAdd(reinterpret_cast<unsigned long long*>(&c->sum_ns), (unsigned long long)d);
  if (D.sums) atomicAdd(&D.sums[(size_t)key * D.S + sig], (unsigned long long)d);
  if (d < *reinterpret_cast<volatile uint64_t*>(&c->min_ns))
    atomicMin(reinterpret_cast<unsigned long long*>(&c->min_ns), (unsigned long long)d);
  if (d > *reinterpret_cast<volatile uint64_t*>(&c->max_ns))
    atomicMax(reinterpret_cast<unsigned long long*>(&c->max_ns), (unsigned long long)d);
  atomicAdd(&c->hist[argus_bucket64(d)], 1u);
  argus_span* sp = reinterpret_cast<argus_span*>(rec + D.span_off) + phase;
  if (start < *reinterpret_cast<volatile int64_t*>(&sp->min_start_ns))
    atomicMin(reinterpret_cast<long long*>(&sp->min_start_ns), (long long)start);
  if (end > *reinterpret_cast<volatile int64_t*>(&sp->max_end_ns))
    atomicMax(reinterpret_cast<long long*>(&sp->max_end_ns), (long long)end);
  atomicAdd(reinterpret_cast<unsigned long long*>(&sp->n_events), 1ull);
}

// Identity bytes of the 16-byte chunk `c` of a record's span+cell area (R7).
// Span area: chunks of argus_span {min_start INT64_MAX, max_end INT64_MIN | span 0, n 0}.
// Cell area: 10 chunks per cell: {count 0, sum 0} {min UINT64_MAX, max 0} then 8 zero hist chunks.
__device__ __forceinline__ uint4 argus_identity_chunk(const argus_dims& D, uint32_t chunk) {
  const uint32_t span_chunks = 2u * (D.P + 1u);
  if (chunk < span_chunks) {
    if (chunk & 1u) return make_uint4(0u, 0u, 0u, 0u);
    return make_uint4(0xFFFFFFFFu, 0x7FFFFFFFu, 0u, 0x80000000u);
  }
  uint32_t part = (chunk - span_chunks) % 10u;
  if (part == 1u) return make_uint4(0xFFFFFFFFu, 0xFFFFFFFFu, 0u, 0u);
  return make_uint4(0u, 0u, 0u, 0u);
}

// The sum-plane row of a record whose cells were just set to their identities.
__device__ __forceinline__ void argus_zero_sums_row(const argus_dims& D, uint32_t key, uint32_t t, uint32_t nt) {
  if (!D.sums) return;
  unsigned long long* row = D.sums + (size_t)key * D.S;
  for (uint32_t i = t; i < D.S; i += nt) row[i] = 0ull;
}

#endif  // __CUDACC__
