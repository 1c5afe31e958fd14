/* argus.h — C ABI of libargus.so: the B200 (sm_100a) hot path of ARGUS
 * (arxiv/paper_2606_20374): kernel-event reduction + cross-rank diagnosis.
 *
 * Citations: "PAPER.md:<line>" is /root/reference/PAPER.md; "NS" is the north_star text of
 * BASELINE.json, which fixes record layouts, the summary contents and the detection rule;
 * "R<n>" is reading n of DESIGN.md §3 (where the paper and NS are silent).
 *
 * This header holds POD layouts and prototypes only: no inline logic.  Every pointer argument is
 * tagged [host] or [device].  Device pointers are plain CUDA global-memory addresses owned by the
 * caller (e.g. torch uint8 tensors); the library borrows them until the work queued on the given
 * stream has completed and never frees them.  `stream` arguments are a `cudaStream_t` passed as
 * `void*` (0 = the legacy default stream).  All functions return ARGUS_OK (0) or a negative
 * ARGUS_E* code; none throws.  Calls on one ctx are not thread-safe.  There is no CPU fallback:
 * without a CUDA device argus_create fails with ARGUS_ECUDA.
 */
#ifndef ARGUS_H_
#define ARGUS_H_

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

/* ---- error codes -------------------------------------------------------------------------- */
#define ARGUS_OK       0
#define ARGUS_EINVAL  -1  /* null / misaligned pointer, zero or out-of-range dimension          */
#define ARGUS_ECUDA   -2  /* a CUDA call failed; see argus_last_cuda_error                      */
#define ARGUS_ESIZE   -3  /* n too large for one call, or dims beyond what the kernels support  */
#define ARGUS_ESTATE  -4  /* call order violated (e.g. aggregate on records that were not reset) */
#define ARGUS_ENOMEM  -5  /* host or device allocation of ctx workspace failed                  */

/* ---- config flags ------------------------------------------------------------------------- */
/* Performance hint (R18): records arrive grouped by (rank, step) — the segmented kernel reads them
 * in place.  Without the hint argus_aggregate first groups the n events of the call by (rank, step)
 * into the grouping area of the workspace (argus_config.max_ungrouped_events * 32 bytes); a call
 * with more events than that area holds takes the slower global-table kernel instead.
 * Results never depend on the hint; a violated hint only costs time. */
#define ARGUS_FLAG_SORTED 0x1u

/* ---- limits ------------------------------------------------------------------------------- */
#define ARGUS_HIST_BUCKETS 32
#define ARGUS_MAX_PHASES   64     /* n_phases <= 64                                              */
#define ARGUS_MAX_RANKS    16384  /* n_ranks  <= 16384 (selection holds one series per CTA)      */

/* ---- flag values written by argus_diagnose (R14) ------------------------------------------ */
#define ARGUS_FLAG_NONE 0
#define ARGUS_FLAG_HIGH 1  /* x > median and |x - median| > 3*MAD */
#define ARGUS_FLAG_LOW  2  /* x < median and |x - median| > 3*MAD */

/* Raw kernel event (NS: "32-byte record {u32 rank, u32 step, u32 sig, u16 stream, u16 phase,
 * i64 start_ns, i64 end_ns}"; the paper's CUPTI activity record — name, launch time, duration,
 * stream — PAPER.md:104, 142).  Little-endian, naturally aligned, no padding (R1). */
typedef struct argus_event {
  uint32_t rank;
  uint32_t step;
  uint32_t sig;      /* interned kernel signature */
  uint16_t stream;   /* carried, not part of the key (R16), not validated (R3) */
  uint16_t phase;
  int64_t  start_ns;
  int64_t  end_ns;
} argus_event;       /* 32 B */

/* Per-(rank, step, sig) summary (NS: "count, u64 sum, min and max of duration, and a 32-bucket
 * log2 duration histogram"; stands where the paper keeps per-cluster (count, p50, p99) triples on
 * a log-duration grid).  Empty cell = reduction identities (R7):
 * count 0, sum 0, min UINT64_MAX, max 0, hist 0.
 * bucket(d) = d==0 ? 0 : min(31, floor(log2 d))  (R4). */
typedef struct argus_cell {
  uint64_t count;
  uint64_t sum_ns;   /* wraps mod 2^64 (R6) */
  uint64_t min_ns;
  uint64_t max_ns;
  uint32_t hist[ARGUS_HIST_BUCKETS];
} argus_cell;        /* 160 B */

/* Per-(rank, step, phase) span and, at index n_phases, the whole-iteration span
 * (NS: "Iteration time is max(end) minus min(start) over a rank-step, and phase time uses the same
 * rule within each phase"; the quantities the paper measures with CUDA events, PAPER.md:128,
 * 222-224).  Empty span (R7): min_start INT64_MAX, max_end INT64_MIN, span 0, n_events 0. */
typedef struct argus_span {
  int64_t  min_start_ns;
  int64_t  max_end_ns;
  uint64_t span_ns;   /* n_events ? max_end - min_start : 0; valid after argus_phase_times */
  uint64_t n_events;
} argus_span;         /* 32 B */

/* Header of the fixed-size per-(rank, step) record (NS (5) "summary encoder that emits the
 * fixed-size per-rank-step record"; R17).  Written by argus_phase_times. */
#define ARGUS_RECORD_MAGIC   0x53475241u /* 'ARGS' little-endian */
#define ARGUS_RECORD_VERSION 1
typedef struct argus_record_header {
  uint32_t magic;
  uint16_t version;
  uint16_t n_phases;
  uint32_t n_sigs;
  uint32_t rank;
  uint32_t step;       /* absolute: step_base + t */
  uint32_t reserved0;  /* 0 */
  uint64_t n_events;   /* = whole span n_events */
  int64_t  min_start_ns;
  int64_t  max_end_ns;
  uint64_t iter_ns;    /* = whole span span_ns */
  uint64_t reserved1;  /* 0 */
} argus_record_header; /* 64 B */

/* Record layout, record (r, t) at byte offset (r*n_steps + t) * argus_record_bytes(cfg):
 *   argus_record_header            64 B
 *   argus_span  span[n_phases + 1] index n_phases = whole iteration
 *   argus_cell  cell[n_sigs]
 */

typedef struct argus_config {
  uint32_t n_ranks;    /* R, 1..ARGUS_MAX_RANKS */
  uint32_t n_steps;    /* T >= 1; a record is addressed by step - step_base in [0, T) (R19);
                          step_base + T <= 2^32 (ARGUS_ESIZE otherwise: step numbers do not wrap) */
  uint32_t n_sigs;     /* S >= 1 */
  uint32_t n_phases;   /* P, 1..ARGUS_MAX_PHASES */
  uint32_t step_base;
  uint32_t flags;      /* ARGUS_FLAG_* */
  int32_t  device;     /* CUDA device ordinal */
  uint32_t max_ungrouped_events; /* largest n of one argus_aggregate call on input WITHOUT the SORTED hint that
                          is still grouped first (sizes the grouping area of the workspace: 32 B per event);
                          0 = no grouping area, ungrouped input goes through the global-table kernel */
  uint32_t max_spill_events; /* RE-QUEUED events the segmented kernel may hold at one time (sizes the spill area of the
                          workspace, 8 B per event, shared evenly by its persistent CTAs): an event whose (rank, step,
                          sig) cell cannot hold it in shared memory — the second mode of a kernel whose durations
                          "differ by several multiples" between positions, PAPER.md:166 — is set aside as {sig, duration}
                          and folded when its rank-step is flushed; 0 or exhausted: such events take L2 reductions
                          one by one (same results, far slower when they are many) */
  uint32_t reserved;   /* 0 */
} argus_config;

/* Per-series result of the cross-rank rule (NS: "per (step, sig), the exact median and MAD over
 * ranks of the u64 summed duration"; R10 median of an even count = lo + (hi-lo)/2). */
typedef struct argus_series_stat {
  uint64_t median;
  uint64_t mad;
  uint32_t n_high;
  uint32_t n_low;
  uint64_t reserved;   /* 0 */
} argus_series_stat;   /* 32 B */

/* Outputs of argus_diagnose: a [host] struct of caller-allocated [device] pointers; any may be
 * NULL to skip that output.  T = n_steps, S = n_sigs, P = n_phases, R = n_ranks. */
typedef struct argus_diag_out {
  argus_series_stat* sig_stats;      /* [T][S]       series x[r] = cell[r][t][s].sum_ns (0 if empty, R11) */
  uint8_t*           sig_flags;      /* [T][S][R]    ARGUS_FLAG_* */
  argus_series_stat* span_stats;     /* [T][P+1]     series x[r] = span[r][t][k].span_ns; k = P whole iteration (R15) */
  uint8_t*           span_flags;     /* [T][P+1][R] */
  uint32_t*          rank_score;     /* [T][R]       # sigs flagged HIGH for (t, r)  — straggler ranks (R15) */
  uint32_t*          step_anomalous; /* [T]          # ranks whose whole-iteration span is HIGH — anomalous steps (R15) */
} argus_diag_out;

typedef struct argus_ctx argus_ctx;  /* opaque */

/* Device workspace of a context, in bytes ("the caller owns every large buffer").  It holds,
 * in this order, each area 256-byte aligned: the per-record state words (4 B per (rank, step)), the event
 * counters, the group sizes of the grouping pass (4 B per (rank, step)), the SUM PLANE (8 B per cell: the
 * u64 sum of every (rank, step, sig), sig-contiguous, kept in step with the table so that the cross-rank
 * gather of argus_diagnose reads whole sectors: 134 MB at R = S = 4096), the per-CTA overflow lists of the
 * segmented kernel (64 KB x 1024), one mark byte per diagnosed series, and — only when
 * cfg->max_ungrouped_events > 0 — the per-CTA key histograms of the grouping pass and the grouping area
 * itself (32 B per event), and — only when cfg->max_spill_events > 0 — the spill area (8 B per event).  Queries the device of cfg for its SM count.  0 if cfg is invalid. */
size_t argus_workspace_bytes(const argus_config* cfg);

/* Create a context for one table geometry.  [device] d_workspace: argus_workspace_bytes(cfg) bytes,
 * 256-byte aligned, owned by the caller, borrowed until argus_destroy (ARGUS_EINVAL when misaligned or
 * workspace_bytes is too small).  d_workspace == NULL: the library makes that one allocation itself, here
 * (ARGUS_ENOMEM when it fails), and frees it in argus_destroy.  No other entry point allocates or frees
 * device memory or synchronises the device.  Host-side the ctx owns an internal copy stream and a few CUDA
 * events.  [host] cfg, [host] out. */
int argus_create(const argus_config* cfg, void* d_workspace, size_t workspace_bytes, argus_ctx** out);
int argus_destroy(argus_ctx* ctx);

/* Bytes of one record = 64 + 32*(P+1) + 160*S, and of the whole [R][T] table.  0 if cfg is NULL. */
size_t argus_record_bytes(const argus_config* cfg);
size_t argus_table_bytes(const argus_config* cfg);

/* Start a new accumulation into [device] d_records (argus_table_bytes, 16-byte aligned).
 * Lazy: marks every record "identity, not yet materialised" in ctx state and zeroes the counters;
 * the table bytes themselves are defined only after argus_phase_times (which materialises the
 * identities of R7 for records no event touched).  Asynchronous on `stream`. */
int argus_reset(argus_ctx* ctx, void* d_records, void* stream);

/* NS (2) ingest: asynchronous copy of n events from [host] pinned memory h_src to [device] d_dst
 * on `copy_stream`, followed by an internal CUDA event that the next argus_aggregate (or
 * argus_aggregate_host) on this ctx waits for, so copy and compute overlap across chunks.  Re-using d_dst
 * while an earlier argus_aggregate may still read it is the caller's business (order copy_stream after
 * the compute stream with an event of your own: see tests/test_ingest_gpu.py).  n may be 0. */
int argus_ingest(argus_ctx* ctx, const argus_event* h_src, uint64_t n, argus_event* d_dst,
                 void* copy_stream);

/* NS (3) aggregate: fold n events at [device] d_events (16-byte aligned; n < 2^32) into the table.
 * May be called repeatedly (chunks may cut rank-steps anywhere; summaries are a monoid, R7).
 * Invalid events (R2: end < start or start < 0; R3: rank/step/sig/phase out of range) are skipped
 * and counted.  Waits for the last argus_ingest.  d_records must be the table given to
 * argus_reset, else ARGUS_ESTATE.  Asynchronous on `stream`. */
int argus_aggregate(argus_ctx* ctx, const argus_event* d_events, uint64_t n, void* d_records,
                    void* stream);

/* NS (2)+(3) streamed aggregate: copy n events from [host] pinned h_events in chunks of
 * chunk_events through a [device] ring of ring_slots slots (each chunk_events*32 bytes; 1..64 slots) on
 * an internal copy stream, overlapped with aggregation of earlier chunks on `stream`.
 * Equivalent to argus_ingest + argus_aggregate per chunk with ring-slot reuse ordered by events: the
 * copy into a slot waits for the aggregation that last read it, the aggregation waits for its copy (the
 * paper's fixed buffer pool with back-pressure; nothing is dropped). */
int argus_aggregate_host(argus_ctx* ctx, const argus_event* h_events, uint64_t n,
                         uint64_t chunk_events, argus_event* d_ring, uint32_t ring_slots,
                         void* d_records, void* stream);

/* Finalise (never re-reads events): materialise untouched records, set every span_ns, derive the
 * whole-iteration span (index P) from the phase spans, write the record headers (NS (5), R17).
 * If [device] d_spans_out is non-NULL also writes a compact copy argus_span[R][T][P+1].
 * Idempotent; may be followed by more argus_aggregate calls and another argus_phase_times (required
 * again before argus_diagnose: ARGUS_ESTATE otherwise). */
int argus_phase_times(argus_ctx* ctx, void* d_records, argus_span* d_spans_out, void* stream);

/* NS (4) cross-rank diagnosis on a finalised table (argus_phase_times must have run since the last
 * argus_aggregate into it, else ARGUS_ESTATE; a table this ctx did not aggregate is read as is).  For every
 * step t and every series family (sigs, phases, whole iteration): exact median and MAD over the
 * R ranks, flag[r] = |x[r]-med| > sat3(MAD) ? (x[r] > med ? HIGH : LOW) : NONE  (R10-R14),
 * plus the roll-ups of R15.  [host] outs holds [device] pointers. */
int argus_diagnose(argus_ctx* ctx, const void* d_records, const argus_diag_out* outs, void* stream);

/* Ownership of a table, made explicit.  "This ctx's table" is the buffer last given to argus_reset, and the
 * library tells it from a foreign one by that address alone: for its own table argus_diagnose takes the sig
 * series from the sum plane of the workspace (kept in step by the aggregation kernels), for any other address
 * it gathers them from the record bytes.  So the bytes of a ctx's table must change only through that ctx.  If
 * the buffer is re-used for other contents (a stored table copied into it, another ctx aggregating into it),
 * call argus_forget first: the ctx then owns no table, argus_diagnose reads every table from its records, and
 * the entry points that need the ctx's own accumulation (argus_aggregate, argus_phase_times, argus_pack_planes)
 * return ARGUS_ESTATE until the next argus_reset.  The encoders, argus_kde_clusters_records and argus_l2_groups
 * read record bytes only: they take any finalised table of the ctx's geometry, forgotten or not.
 * Skipping it is a usage error the library cannot detect: medians and flags of the sig series would come from
 * the stale sum plane while the spans come from the new bytes.  Host-side only; queues nothing. */
int argus_forget(argus_ctx* ctx);

/* ---- one job sharded by trace rank over several GPUs (the paper's comparison of "the same
 * kernel across different ranks", when the ranks' events live on different devices) --------
 * Every GPU g aggregates its own ranks [r0_g, r0_g + R_g) with a ctx of n_ranks = R_g (events carry
 * rank - r0_g).  Aggregation and spans need no exchange.  The cross-rank rule needs, per (step, series),
 * the value of EVERY rank: the one exchange is the 8-byte-per-cell sum plane (and the tiny span plane),
 * transposed so that GPU d owns a slice of the sigs for ALL ranks:
 *     sig plane  of a slice [s0, s1):  x[r] of series (t, s) at  plane[((t*(s1-s0) + (s-s0)) * rank_stride + r]
 *     span plane:                      x[r] of series (t, k) at  plane[((t*(P+1) + k) * rank_stride + r]
 * argus_pack_planes writes this ctx's ranks into columns [rank_offset, rank_offset + R_g) of such planes;
 * the destination may be local memory (a send buffer for an all-to-all: rank_stride = R_g, rank_offset = 0)
 * or the owning peer's plane mapped over NVLink (rank_stride = R, rank_offset = r0_g: the exchange is then
 * the kernel's own coalesced stores, rows of R_g contiguous u64).  argus_diagnose_planes runs the rule
 * of argus_diagnose on planes; rank_score comes out as the partial count over the slice's sigs (sum the
 * partials of all slices), every other output is final for the series of the slice. */
typedef struct argus_planes {
  const uint64_t* sig_sums;    /* [device] [T][n_sigs][rank_stride] u64 summed durations (0 = empty cell, R11), or NULL */
  const uint64_t* span_ns;     /* [device] [T][P+1][rank_stride]    u64 span_ns, or NULL */
  uint32_t n_ranks;            /* R of the whole job, 1..ARGUS_MAX_RANKS */
  uint32_t rank_stride;        /* >= n_ranks, in elements */
  uint32_t n_sigs;             /* sigs of this slice (0 with sig_sums == NULL); <= cfg.n_sigs of the ctx */
  uint32_t reserved;           /* 0 */
} argus_planes;

/* Export sigs [sig_lo, sig_hi) of this ctx's finalised table (argus_phase_times ran; ARGUS_ESTATE otherwise)
 * into [device] planes as laid out above.  d_sig_plane and/or d_span_plane may be NULL to skip.
 * 8-byte aligned; rank_offset + cfg.n_ranks <= rank_stride.  Asynchronous on `stream`. */
int argus_pack_planes(argus_ctx* ctx, const void* d_records, uint32_t sig_lo, uint32_t sig_hi,
                      uint64_t* d_sig_plane, uint64_t* d_span_plane, uint32_t rank_stride,
                      uint32_t rank_offset, void* stream);

/* The cross-rank rule (R10-R15) on planes: outs->sig_stats [T][n_sigs], sig_flags [T][n_sigs][R],
 * span_stats [T][P+1], span_flags [T][P+1][R], rank_score [T][R] (partial: this slice's sigs),
 * step_anomalous [T]; T and P are the ctx's, R = planes->n_ranks.  [host] planes, [host] outs. */
int argus_diagnose_planes(argus_ctx* ctx, const argus_planes* planes, const argus_diag_out* outs, void* stream);

/* The same rule for callers that must not allocate device memory: no ctx, no workspace, no cudaMalloc /
 * cudaFree / allocating library call anywhere on this path.  Who that is: a monitor living inside the training
 * process it observes (the paper's collector is injected into the job and reuses pre-allocated buffers) — the framework's
 * caching allocator has usually claimed the HBM already, so a cudaMalloc from the side can fail outright, and
 * when it succeeds it takes a device-wide lock and may stall the very iteration being measured; the same goes
 * for code that runs from a callback or another context in which the CUDA runtime forbids allocation.  Such a
 * caller hands in buffers it carved out at start-up (planes and outputs, exactly as for
 * argus_diagnose_planes) and this entry point supplies the one piece of scratch the selection needs — a mark
 * byte per series, set by the 32-bit pass for the series the 64-bit pass must redo — from a fixed array that
 * is part of the library image: ARGUS_STATIC_MAX_SERIES bytes (256 KiB) of global memory on every device that
 * loads libargus.so, held until the process exits.
 *   n_steps = T >= 1, n_phases = P in 1..ARGUS_MAX_PHASES (what the ctx would have carried);
 *   T * (planes->n_sigs + P + 1) series must fit the array, else ARGUS_ESIZE and nothing is launched.
 * Works on the CURRENT device of the calling thread, which must be the one that holds the buffers.  The first
 * call on each device looks up the array's device address and the SM count (host-side, once, under a lock):
 * make that first call outside any stream capture.  Every call on a device shares the one array and leaves
 * its marks behind; each call clears the bytes it is about to use on `stream` first, so calls ordered on one
 * stream (or by events) are independent, but two calls that can overlap on the same device race on the marks
 * and may return wrong medians for series whose values span 2^32 ns or more — serialise them.  Outputs and
 * errors as argus_diagnose_planes (ARGUS_EINVAL for more than ARGUS_STATIC_MAX_DEVICES device ordinals). */
#define ARGUS_STATIC_MAX_SERIES  262144u
#define ARGUS_STATIC_MAX_DEVICES 64
int argus_diagnose_planes_static(const argus_planes* planes, uint32_t n_steps, uint32_t n_phases,
                                 const argus_diag_out* outs, void* stream);

/* ---- compact record encodings (second half: "sparse/bit-packed record encoding (non-empty
 * bins only) to raise the compression ratio"; the paper's per-rank record of "approximately 200 triples ... about
 * 2.7 KB").  Both turn this ctx's FINALISED table (argus_phase_times ran; ARGUS_ESTATE otherwise)
 * into one byte stream of variable-length records in (rank, step) order; every field little-endian, every part
 * 8-byte aligned.  Record k occupies [d_offsets[k], d_offsets[k+1]) of d_out; d_offsets[R*T] = total length.
 *   SPARSE (R37, lossless):
 *     argus_record_header   version = 2, reserved0 = number of non-empty cells, reserved1 = byte length of the record
 *     u64 phase_mask        bit k: phase span k (k < P) has n_events != 0 (the whole-iteration span is in the header)
 *     argus_span            one per set bit, ascending k
 *     per non-empty cell (count != 0), ascending sig:
 *       u32 sig | u8 b0 | u8 nb | u16 0         b0 = bucket(min_ns), nb = bucket(max_ns) - b0 + 1
 *       u64 count | u64 sum_ns | u64 min_ns | u64 max_ns
 *       u32 hist[b0 .. b0 + nb) | u32 0 when nb is odd
 *   TRIPLE (R38, the paper's (count, p50, p99) record; lossy: what NEXT-1 keeps of a cell):
 *     argus_record_header   version = 3, reserved0 = number of cells with >= 1 cluster, reserved1 = byte length
 *     u64 phase_mask + spans as above
 *     per cell with n_clusters > 0, ascending sig:  u32 sig | u32 n_clusters | n_clusters x argus_cluster
 * [device] d_out (8-byte aligned, out_capacity bytes), [device] d_offsets [R*T + 1] u64.  A record that would end
 * beyond out_capacity is not written (d_offsets is still complete: compare d_offsets[R*T] with out_capacity);
 * argus_sparse_bound / argus_triple_bound give a capacity that always suffices.  Asynchronous on `stream`.
 * The encoders of ONE ctx share a ticket word in its workspace, cleared by every call: two encodes of the same
 * ctx (sparse and triple, or two of a kind) must not overlap on the GPU — queue them on one stream or order them
 * with events, else records are handed out twice and the look-back never completes.  Different ctxs are
 * independent.  TRIPLE: a d_n_clusters entry larger than max_clusters is read as max_clusters. */
size_t argus_sparse_bound(const argus_config* cfg);
int argus_sparse_encode(argus_ctx* ctx, const void* d_records, uint8_t* d_out, uint64_t out_capacity,
                        uint64_t* d_offsets, void* stream);

/* ==== the paper's own float algorithms (SURVEY 8(f) NEXT-1..3), fp64; every constant the paper leaves open
 * is a parameter whose default is a reading of DESIGN.md 3 (R23-R36) ================================== */

/* ---- NEXT-1: online statistical compression (eq. 1) ---------------------------------
 * "applies a logarithmic transformation to the raw durations, then computes the KDE density function on an
 * equally-spaced grid" with Scott's bandwidth, "local minima (valleys) as cluster boundaries", two filters,
 * then "(count, p50, p99)" per cluster.  The grid is a histogram of log-durations with per_octave bins per
 * factor of two: the 32-bucket histogram of the records (per_octave = 1), or the fine histogram of
 * argus_fine_hist (per_octave = 8, 256 bins: bin(d) = floor(8 log2 d), 0 for d <= 1, 255 for d >= 2^32). */
typedef struct argus_cluster {
  uint32_t count;      /* 0 = unused slot */
  uint16_t p50_bin;    /* grid bin where the cluster's cumulative count first reaches ceil(0.5 count) */
  uint16_t p99_bin;    /* ... ceil(0.99 count); a bin stands for 2^((bin + 0.5) / per_octave) ns */
} argus_cluster;       /* 8 B */
typedef struct argus_kde_params {
  uint32_t per_octave;    /* grid steps per factor of two: 1 or 8 */
  uint32_t n_bins;        /* 32 or 256 (<= 256) */
  uint32_t min_count;     /* cluster-level filter: both sides of a kept valley hold >= max(min_count, min_frac n) samples (8) */
  uint32_t min_gap_bins;  /* spacing filter: kept boundaries are >= this many grid steps apart (half an octave) */
  uint32_t max_clusters;  /* output slots per cell (the last one takes the rest), 1..16 */
  uint32_t reserved;
  double   min_frac;      /* 0.02 */
} argus_kde_params;
/* Fine histogram of the valid events' durations per (rank, step, sig): [device] d_hist [R][T][S][256] u32,
 * accumulated into (the caller zeroes it).  L2 atomics: meant for the sizes a [R][T][S][256] table fits. */
int argus_fine_hist(argus_ctx* ctx, const argus_event* d_events, uint64_t n, uint32_t* d_hist, void* stream);
/* n_cells histograms of p->n_bins counters -> [device] d_clusters [n_cells][max_clusters], d_n_clusters
 * [n_cells]; d_density [n_cells][n_bins] f64 receives the density of eq. (1) (with 1/h) or may be NULL. */
int argus_kde_clusters(argus_ctx* ctx, const uint32_t* d_hist, uint64_t n_cells, const argus_kde_params* p,
                       argus_cluster* d_clusters, uint8_t* d_n_clusters, double* d_density, void* stream);
/* The same on the 32-bucket histograms of this ctx's finalised record table (p->per_octave = 1, n_bins = 32):
 * d_clusters [R][T][S][max_clusters], d_n_clusters [R][T][S].  No pass over the events. */
int argus_kde_clusters_records(argus_ctx* ctx, const void* d_records, const argus_kde_params* p,
                               argus_cluster* d_clusters, uint8_t* d_n_clusters, void* stream);

/* The TRIPLE record stream (layout above) from the clusters of argus_kde_clusters(_records) over this ctx's
 * table: [device] d_clusters [R][T][S][max_clusters], d_n_clusters [R][T][S]. */
size_t argus_triple_bound(const argus_config* cfg, uint32_t max_clusters);
int argus_triple_encode(argus_ctx* ctx, const void* d_records, const argus_cluster* d_clusters,
                        const uint8_t* d_n_clusters, uint32_t max_clusters, uint8_t* d_out, uint64_t out_capacity,
                        uint64_t* d_offsets, void* stream);

/* ---- NEXT-2: L3 kernel-statistics anomaly detection (eq. 2-4) -------------------------
 * Per key (kernel): every rank's clusters (count, p50, p99) -> log-normal mixture CDF (mu = ln p50,
 * sigma = (ln p99 - ln p50)/2.326) on a log-uniform grid of n_grid points from 0.5 min p50 to 2 max p99 ->
 * W1 by the trapezoid rule -> score = mean W1 to the other ranks -> flag when score > Q3 + alpha (Q3 - Q1). */
typedef struct argus_l3_in {
  const uint32_t* count;   /* [device] [n_keys][n_ranks][max_clusters] (0 = no cluster) */
  const double*   p50;     /* [device] same shape, ns */
  const double*   p99;
  uint32_t n_keys, n_ranks /* <= 4096 */, max_clusters, reserved;
} argus_l3_in;
typedef struct argus_l3_params { uint32_t n_grid /* >= 2 (256) */; uint32_t reserved; double alpha /* 1.5 */; } argus_l3_params;
typedef struct argus_l3_stat { double q1, q3, fence, x_lo, x_hi; } argus_l3_stat;
/* The clusters of argus_kde_clusters(_records) over this ctx's table, [R][T][S][max_clusters], regrouped as
 * the L3 input of key (t, s): [device] d_count / d_p50 / d_p99 [T*S][R][max_clusters]; a bin becomes the
 * duration it stands for, 2^((bin + 0.5) / per_octave) ns (R30). */
int argus_clusters_to_l3(argus_ctx* ctx, const argus_cluster* d_clusters, uint32_t max_clusters, uint32_t per_octave,
                         uint32_t* d_count, double* d_p50, double* d_p99, void* stream);
/* [device] d_score [n_keys][n_ranks] f64, d_stat [n_keys], d_flags [n_keys][n_ranks] u8. */
int argus_l3_detect(argus_ctx* ctx, const argus_l3_in* in, const argus_l3_params* p, double* d_score,
                    argus_l3_stat* d_stat, uint8_t* d_flags, void* stream);

/* ---- NEXT-3: L2 phase-level attribution (eq. 5, Table 3) ---------------------
 * For every phase span k (index P = whole iteration) of this ctx's finalised table: x_r = mean over the T
 * steps of span_ns; the ranks are compared inside the parallelism group the event is routed to:
 * d_route [P+1] u8 names the dimension of event k, d_group_id [n_dims][R] u32 the group (an id < R; >= R =
 * none) of every rank in each dimension.  Per group: n, mu, sigma (|G| - 1), CV = sigma/mu and its class
 * (0 balanced < 0.02 <= 1 mild < 0.05 <= 2 severe); per rank z = (x - mu)/sigma, flag = z > z_threshold. */
typedef struct argus_l2_group { uint32_t n, cls; double mu, sigma, cv; } argus_l2_group;   /* 32 B */
/* [device] d_groups [P+1][R] (indexed by group id; n = 0: no such group), d_z [P+1][R] f64, d_flags [P+1][R]
 * u8, d_xbar [P+1][R] f64 (the x_r; also scratch).  n_dims in 1..256 is the first extent of d_group_id; an
 * event whose route byte is >= n_dims joins no group (z = 0, no flag, no group entries) rather than reading past
 * the array.  Group sums are taken in a fixed order (no floating-point atomics): results are the same bits in
 * every run, so a CV class or a z flag cannot flip between runs. */
int argus_l2_groups(argus_ctx* ctx, const void* d_records, const uint8_t* d_route, uint32_t n_dims,
                    const uint32_t* d_group_id, double z_threshold, argus_l2_group* d_groups, double* d_z, uint8_t* d_flags, double* d_xbar,
                    void* stream);

/* ---- NEXT-3: L1 iteration-level detection ----------------------------------------------
 * n_series time series of n_steps u64 values (iteration times in ns), value (s, t) at
 * d_base + s*series_stride + t*step_stride bytes (e.g. the span_ns of index P in argus_phase_times'
 * d_spans_out).  Jitter: windows of `window` points whose max/min exceeds theta are candidates, adjacent or
 * overlapping ones merge; per merged interval the baseline is the median of the points outside it and the
 * effective width the longest run inside it above beta x baseline.  Change point: the split (both sides >=
 * min_seg points) with the largest mu_R/mu_L among those with mu_R/mu_L > ratio_min and sigma/mu < rsd_max on
 * both sides.  cls: 0 stable, 1 jitter, 2 regression, 3 both.  n_steps <= 2048. */
#define ARGUS_L1_MAX_INTERVALS 8
typedef struct argus_l1_params {
  uint32_t window /* 8 */, min_seg /* 4 */;
  double theta /* 1.5 */, beta /* 1.25 */, ratio_min /* 1.1 */, rsd_max /* 0.05 */;
} argus_l1_params;
typedef struct argus_l1_interval { uint32_t first, last, width, reserved; double baseline; } argus_l1_interval;  /* 24 B */
typedef struct argus_l1_out {
  uint32_t cls, n_intervals /* may exceed ARGUS_L1_MAX_INTERVALS: only the first are stored */, cp_found, cp_step;
  double cp_ratio;
  argus_l1_interval interval[ARGUS_L1_MAX_INTERVALS];
} argus_l1_out;
int argus_l1_detect(argus_ctx* ctx, const void* d_base, uint64_t series_stride, uint64_t step_stride,
                    uint32_t n_series, uint32_t n_steps, const argus_l1_params* p, argus_l1_out* d_out, void* stream);

/* Synchronises the internal copy stream and every stream passed to this ctx since argus_create (the ctx
 * remembers up to 8 distinct ones; the oldest is synchronised when a ninth appears) and returns the event
 * counters since argus_reset.  Asynchronous kernel faults surface here as ARGUS_ECUDA.  [host] outputs,
 * may be NULL. */
int argus_stats(argus_ctx* ctx, uint64_t* n_valid, uint64_t* n_invalid);

/* Events the shared-memory compact cells of the segmented kernel refused since argus_reset (duration >= 2^32
 * ns, or a (rank, step, sig) whose durations spread over more than four consecutive log2 buckets: heavy
 * tails, multimodal kernels): n_requeued went through the spill area and were folded at the flush of their rank-step,
 * n_overflow took the overflow list / L2 reductions.  A throughput diagnostic: results do not depend on
 * it.  Synchronises like argus_stats.  [host] outputs, may be NULL. */
int argus_refused_count(argus_ctx* ctx, uint64_t* n_requeued, uint64_t* n_overflow);

/* Keys argus_l3_detect has scored since argus_reset, by the way the kernel took: n_class = the ranks of the key
 * fell into at most 256 classes of identical mixtures (the score is a weighted sum over classes), n_general = more
 * distinct mixtures than that (a sort of the R CDF values per grid point; about an order of magnitude slower per
 * key), n_empty = no rank had a cluster.  A throughput diagnostic: results do not depend on the path.
 * Synchronises like argus_stats.  [host] outputs, may be NULL. */
int argus_l3_path_count(argus_ctx* ctx, uint64_t* n_class, uint64_t* n_general, uint64_t* n_empty);

/* Kernels and memsets this ctx has launched since argus_create (what bench.py reports as gpu_launches).
 * [host] outputs, may be NULL. */
int argus_launch_count(const argus_ctx* ctx, uint64_t* kernels, uint64_t* memsets);

/* Knobs for tests and measurement (not needed for correctness): which = ARGUS_TUNE_*.  */
#define ARGUS_TUNE_GRID_CTAS   1  /* persistent CTAs of the segmented kernel (0 = by geometry; <= 1024) */
#define ARGUS_TUNE_FORCE_PATH  2  /* 0 = by flags, 1 = segmented, 2 = global-table, 3 = group then segmented */
int argus_tune(argus_ctx* ctx, int which, int64_t value);

const char* argus_strerror(int code);
int         argus_last_cuda_error(const argus_ctx* ctx); /* cudaError_t of the last ARGUS_ECUDA */
const char* argus_version(void);

#ifdef __cplusplus
}
#endif
#endif /* ARGUS_H_ */
