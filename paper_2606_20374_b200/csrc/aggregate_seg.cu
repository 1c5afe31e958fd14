// aggregate_seg.cu — segmented aggregation kernel (NS (3): "hand-written sm_100a aggregation
// kernels ... coalesced 128-bit vectorised loads, with TMA ... staging into shared memory ...
// shared-memory-privatised per-block histograms and min/max/sum ... warp-shuffle segmented
// reductions where a block spans rank-step boundaries, and flush to global in one pass").
//
// One persistent CTA per SM walks a contiguous span of the event buffer.  Events arrive through a
// ring of 8 KB stages filled by 1-D TMA bulk copies (cp.async.bulk + mbarrier complete_tx).  The
// CTA keeps ONE (rank, step) table in shared memory at a time, in a compact 32-byte cell per sig
// (DESIGN.md §6.1): four tagged histogram slots {bucket+1 : 6 bits | count : 26 bits}, a 64-bit
// sum split into two u32 words with carry, ~min and max as u32.  Only native 32-bit shared atomics
// are used (64-bit shared atomics compile to CAS loops on sm_100a).  An event the compact cell
// cannot take (duration >= 2^32 ns, or a fifth distinct bucket of one sig) goes straight to the
// global record with L2 atomics.  When the (rank, step) key changes the table is flushed: the
// first CTA to reach a record claims it and writes the whole 160-byte cells with coalesced
// 128-bit stores (no read-modify-write, no separate identity fill); any later contribution to the
// same record merges with L2 reductions.  Correct for ANY event order; fast when events are
// grouped by (rank, step) (R18).
#include "argus_internal.cuh"

namespace {

constexpr int NT = 1024;             // threads per CTA
constexpr int SUB = 256;             // events per TMA stage (8 KB)
constexpr int G = NT / SUB;          // stages consumed per iteration
constexpr int MAXK = 20;             // ring stages (bounded by shared memory at launch)
constexpr uint32_t KEY_NONE = 0xFFFFFFFFu;
constexpr uint32_t FULL = 0xFFFFFFFFu;
constexpr int HDR_BYTES = 256;
constexpr int SPAN_BYTES = ARGUS_MAX_PHASES * 32;

struct SpanAcc {                      // shared-memory span accumulator of one phase (32 B)
  long long mn, mx;
  unsigned long long n;
  unsigned long long pad;
};

struct Hdr {
  unsigned long long bars[MAXK];      // mbarriers, one per stage
  uint32_t cur_key;
  uint32_t flags;                     // bit 0: some event of this iteration needs the global path
  uint32_t next_idx;                  // lowest pending event index (key switch)
  uint32_t mode;                      // state word seen by the flush claim
};
static_assert(sizeof(Hdr) <= HDR_BYTES, "header");

__device__ __forceinline__ uint32_t smem_u32(const void* p) {
  return (uint32_t)__cvta_generic_to_shared(p);
}
__device__ __forceinline__ void mbar_init(uint32_t bar, uint32_t count) {
  asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(bar), "r"(count));
}
__device__ __forceinline__ void mbar_expect_tx(uint32_t bar, uint32_t bytes) {
  asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(bar), "r"(bytes)
               : "memory");
}
__device__ __forceinline__ void tma_load_1d(uint32_t dst, const void* src, uint32_t bytes,
                                            uint32_t bar) {
  asm volatile(
      "cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];" ::"r"(dst),
      "l"(src), "r"(bytes), "r"(bar)
      : "memory");
}
__device__ __forceinline__ void mbar_wait(uint32_t bar, uint32_t parity) {
  asm volatile(
      "{\n"
      ".reg .pred P1;\n"
      "LAB_WAIT:\n"
      "mbarrier.try_wait.parity.shared::cta.b64 P1, [%0], %1;\n"
      "@P1 bra DONE;\n"
      "bra LAB_WAIT;\n"
      "DONE:\n"
      "}" ::"r"(bar),
      "r"(parity)
      : "memory");
}

__device__ __forceinline__ long long warp_min_i64(long long v) {
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) {
    long long w = __shfl_xor_sync(FULL, v, o);
    v = w < v ? w : v;
  }
  return v;
}
__device__ __forceinline__ long long warp_max_i64(long long v) {
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) {
    long long w = __shfl_xor_sync(FULL, v, o);
    v = w > v ? w : v;
  }
  return v;
}

// Per-warp register accumulator of one phase's span (the common case: 32 consecutive events of a
// warp share key and phase).
struct WarpSpan {
  uint32_t phase;  // warp-uniform; KEY_NONE = empty
  uint32_t n;
  long long mn, mx;
  __device__ __forceinline__ void reset() {
    phase = KEY_NONE; n = 0; mn = INT64_MAX; mx = INT64_MIN;
  }
  // all 32 lanes call
  __device__ __forceinline__ void flush(SpanAcc* spans, int lane) {
    if (phase != KEY_NONE) {
      long long a = warp_min_i64(mn), b = warp_max_i64(mx);
      uint32_t c = __reduce_add_sync(FULL, n);
      if (lane == 0 && c) {
        atomicMin(&spans[phase].mn, a);
        atomicMax(&spans[phase].mx, b);
        atomicAdd(&spans[phase].n, (unsigned long long)c);
      }
    }
    reset();
  }
};

struct Ctx {
  Hdr* H;
  SpanAcc* spans;
  uint4* table;  // 2 uint4 per sig: {slot0..3} {sum_lo, sum_hi, ~min, max}
  uint8_t* records;
  uint32_t* state;
  argus_dims D;
};

// Fold one accepted event into the compact table.  Returns false if it needs the global path.
__device__ __forceinline__ bool cell_accumulate(uint4* table, uint32_t sig, uint64_t d) {
  if (d >> 32) return false;
  const uint32_t d32 = (uint32_t)d;
  const uint32_t tag = (31u - (uint32_t)__clz((int)(d32 | 1u))) + 1u;  // bucket + 1, 1..32
  uint32_t* cell = reinterpret_cast<uint32_t*>(table + 2 * sig);
  const uint4 s = *reinterpret_cast<const uint4*>(cell);
  int j = -1;
  if ((s.x & 63u) == tag) j = 0;
  else if ((s.y & 63u) == tag) j = 1;
  else if ((s.z & 63u) == tag) j = 2;
  else if ((s.w & 63u) == tag) j = 3;
  if (j >= 0) {
    atomicAdd(cell + j, 64u);
  } else {
    // claim a slot (first events of a sig in this rank-step); slots fill in order and are never
    // released before the flush, so a tag lives in at most one slot
    bool done = false;
#pragma unroll 1
    for (int k = 0; k < 4 && !done; ++k) {
      uint32_t v = *reinterpret_cast<volatile uint32_t*>(cell + k);
      if (v == 0u) {
        v = atomicCAS(cell + k, 0u, tag | 64u);
        if (v == 0u) { done = true; break; }
      }
      if ((v & 63u) == tag) { atomicAdd(cell + k, 64u); done = true; }
    }
    if (!done) return false;
  }
  const uint32_t old = atomicAdd(cell + 4, d32);
  if (old + d32 < old) atomicAdd(cell + 5, 1u);
  const uint2 mm = *reinterpret_cast<const uint2*>(cell + 6);
  if (~d32 > mm.x) atomicMax(cell + 6, ~d32);
  if (d32 > mm.y) atomicMax(cell + 7, d32);
  return true;
}

// 16-byte chunk `part` (0..9) of the 160-byte argus_cell decoded from a compact cell.
__device__ __forceinline__ uint4 cell_chunk(const uint4 s, const uint4 m, uint32_t part) {
  const uint32_t c0 = s.x >> 6, c1 = s.y >> 6, c2 = s.z >> 6, c3 = s.w >> 6;
  if (part == 0u) {
    unsigned long long cnt = (unsigned long long)c0 + c1 + c2 + c3;
    return make_uint4((uint32_t)cnt, (uint32_t)(cnt >> 32), m.x, m.y);
  }
  if (part == 1u) {
    if ((c0 | c1 | c2 | c3) == 0u) return make_uint4(0xFFFFFFFFu, 0xFFFFFFFFu, 0u, 0u);
    return make_uint4(~m.z, 0u, m.w, 0u);
  }
  const uint32_t b0 = 4u * (part - 2u) + 1u;  // tag of the chunk's first bucket
  const uint32_t t0 = s.x & 63u, t1 = s.y & 63u, t2 = s.z & 63u, t3 = s.w & 63u;
  uint4 v;
  v.x = (t0 == b0 ? c0 : 0u) + (t1 == b0 ? c1 : 0u) + (t2 == b0 ? c2 : 0u) + (t3 == b0 ? c3 : 0u);
  v.y = (t0 == b0 + 1 ? c0 : 0u) + (t1 == b0 + 1 ? c1 : 0u) + (t2 == b0 + 1 ? c2 : 0u) + (t3 == b0 + 1 ? c3 : 0u);
  v.z = (t0 == b0 + 2 ? c0 : 0u) + (t1 == b0 + 2 ? c1 : 0u) + (t2 == b0 + 2 ? c2 : 0u) + (t3 == b0 + 2 ? c3 : 0u);
  v.w = (t0 == b0 + 3 ? c0 : 0u) + (t1 == b0 + 3 ? c1 : 0u) + (t2 == b0 + 3 ? c2 : 0u) + (t3 == b0 + 3 ? c3 : 0u);
  return v;
}

// Flush the shared table of record `key` to global memory and clear it.  All threads call.
// The caller has flushed its WarpSpan first.
__device__ __noinline__ void flush_table(const Ctx& c, uint32_t key) {
  const int tid = threadIdx.x;
  const argus_dims& D = c.D;
  __syncthreads();
  if (tid == 0) {
    uint32_t old = atomicCAS(&c.state[key], ARGUS_ST_LAZY, ARGUS_ST_BUSY);
    if (old == ARGUS_ST_BUSY) {
      // another (resident, running) CTA is writing this record: wait for it, then merge
      while (atomicAdd(&c.state[key], 0u) != ARGUS_ST_LIVE) __nanosleep(128);
      __threadfence();
      old = ARGUS_ST_LIVE;
    }
    c.H->mode = old;
  }
  __syncthreads();
  const uint32_t mode = c.H->mode;
  uint8_t* rec = c.records + (size_t)key * D.rec_bytes;
  if (mode == ARGUS_ST_LAZY) {
    // we own the record: write spans + cells once, coalesced 16-byte chunks
    uint4* dst = reinterpret_cast<uint4*>(rec + D.span_off);
    const uint32_t span_chunks = 2u * (D.P + 1u);
    const uint32_t n_chunks = span_chunks + 10u * D.S;
    for (uint32_t ch = tid; ch < n_chunks; ch += NT) {
      uint4 v;
      if (ch < span_chunks) {
        const uint32_t k = ch >> 1;
        if (k < D.P && c.spans[k].n != 0ull) {
          const SpanAcc a = c.spans[k];
          v = (ch & 1u) ? make_uint4(0u, 0u, (uint32_t)a.n, (uint32_t)(a.n >> 32))
                        : make_uint4((uint32_t)a.mn, (uint32_t)((unsigned long long)a.mn >> 32),
                                     (uint32_t)a.mx, (uint32_t)((unsigned long long)a.mx >> 32));
        } else {
          v = argus_identity_chunk(D, ch);
        }
      } else {
        const uint32_t cc = ch - span_chunks;
        const uint32_t sig = cc / 10u, part = cc - sig * 10u;
        v = cell_chunk(c.table[2 * sig], c.table[2 * sig + 1], part);
      }
      dst[ch] = v;
    }
    __threadfence();
    __syncthreads();
    if (tid == 0) atomicExch(&c.state[key], ARGUS_ST_LIVE);
  } else {
    // merge into a live record with L2 reductions (non-empty fields only)
    argus_cell* cells = reinterpret_cast<argus_cell*>(rec + D.cell_off);
    for (uint32_t sig = tid; sig < D.S; sig += NT) {
      const uint4 s = c.table[2 * sig], m = c.table[2 * sig + 1];
      const uint32_t sl[4] = {s.x, s.y, s.z, s.w};
      unsigned long long cnt = 0;
#pragma unroll
      for (int k = 0; k < 4; ++k) {
        const uint32_t ck = sl[k] >> 6;
        if (ck) {
          atomicAdd(&cells[sig].hist[(sl[k] & 63u) - 1u], ck);
          cnt += ck;
        }
      }
      if (cnt) {
        atomicAdd(reinterpret_cast<unsigned long long*>(&cells[sig].count), cnt);
        atomicAdd(reinterpret_cast<unsigned long long*>(&cells[sig].sum_ns),
                  ((unsigned long long)m.y << 32) | m.x);
        atomicMin(reinterpret_cast<unsigned long long*>(&cells[sig].min_ns),
                  (unsigned long long)(~m.z));
        atomicMax(reinterpret_cast<unsigned long long*>(&cells[sig].max_ns),
                  (unsigned long long)m.w);
      }
    }
    argus_span* sp = reinterpret_cast<argus_span*>(rec + D.span_off);
    for (uint32_t k = tid; k < D.P; k += NT) {
      const SpanAcc a = c.spans[k];
      if (a.n) {
        atomicMin(reinterpret_cast<long long*>(&sp[k].min_start_ns), a.mn);
        atomicMax(reinterpret_cast<long long*>(&sp[k].max_end_ns), a.mx);
        atomicAdd(reinterpret_cast<unsigned long long*>(&sp[k].n_events), a.n);
      }
    }
  }
  __syncthreads();
  for (uint32_t i = tid; i < 2u * D.S; i += NT) c.table[i] = make_uint4(0u, 0u, 0u, 0u);
  for (uint32_t k = tid; k < D.P; k += NT) {
    c.spans[k].mn = INT64_MAX; c.spans[k].mx = INT64_MIN; c.spans[k].n = 0ull; c.spans[k].pad = 0ull;
  }
  __syncthreads();
}

__global__ void __launch_bounds__(NT, 1)
aggregate_seg_kernel(const uint4* __restrict__ ev, uint64_t n, uint64_t per_cta, uint8_t* records,
                     uint32_t* state, unsigned long long* counters, argus_dims D, int K) {
  extern __shared__ __align__(128) uint8_t smem[];
  Ctx c;
  c.H = reinterpret_cast<Hdr*>(smem);
  c.spans = reinterpret_cast<SpanAcc*>(smem + HDR_BYTES);
  c.table = reinterpret_cast<uint4*>(smem + HDR_BYTES + SPAN_BYTES);
  c.records = records; c.state = state; c.D = D;
  uint8_t* stages = smem + ((HDR_BYTES + SPAN_BYTES + 32u * D.S + 127u) & ~127u);

  const int tid = threadIdx.x, lane = tid & 31;
  const uint64_t e0 = (uint64_t)blockIdx.x * per_cta;
  if (e0 >= n) return;
  const uint64_t e1 = (e0 + per_cta < n) ? e0 + per_cta : n;
  const uint32_t n_ev = (uint32_t)(e1 - e0);
  const uint32_t n_sub = (n_ev + SUB - 1) / SUB;
  const uint32_t n_iter = (n_ev + NT - 1) / NT;
  const uint4* src = ev + 2 * e0;

  if (tid == 0) {
    for (int k = 0; k < K; ++k) mbar_init(smem_u32(&c.H->bars[k]), 1u);
    c.H->cur_key = KEY_NONE; c.H->flags = 0u; c.H->next_idx = KEY_NONE; c.H->mode = 0u;
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
  }
  for (uint32_t i = tid; i < 2u * D.S; i += NT) c.table[i] = make_uint4(0u, 0u, 0u, 0u);
  for (uint32_t k = tid; k < ARGUS_MAX_PHASES; k += NT) {
    c.spans[k].mn = INT64_MAX; c.spans[k].mx = INT64_MIN; c.spans[k].n = 0ull; c.spans[k].pad = 0ull;
  }
  __syncthreads();

  auto issue = [&](uint32_t s) {  // thread 0 only
    const uint32_t slot = s % (uint32_t)K;
    const uint32_t cnt = (n_ev - s * SUB < (uint32_t)SUB) ? n_ev - s * SUB : (uint32_t)SUB;
    const uint32_t bar = smem_u32(&c.H->bars[slot]);
    mbar_expect_tx(bar, cnt * 32u);
    tma_load_1d(smem_u32(stages + (size_t)slot * SUB * 32), src + 2 * (size_t)s * SUB, cnt * 32u, bar);
  };
  if (tid == 0)
    for (uint32_t s = 0; s < (uint32_t)K && s < n_sub; ++s) issue(s);

  WarpSpan ws;
  ws.reset();
  uint32_t cur_key = KEY_NONE;
  uint32_t n_valid = 0, n_invalid = 0;

  for (uint32_t it = 0; it < n_iter; ++it) {
    const uint32_t s = it * G + (uint32_t)(tid / SUB);
    const uint32_t idx = it * NT + (uint32_t)tid;
    const bool active = idx < n_ev;
    uint32_t rank = 0, step = 0, sig = 0, phase = 0, key = KEY_NONE;
    long long start = 0, end = 0;
    bool pending = false;
    if (s < n_sub) {
      mbar_wait(smem_u32(&c.H->bars[s % (uint32_t)K]), (s / (uint32_t)K) & 1u);
      if (active) {
        // lanes 0-3,8-11,.. read the first half first, the others the second: conflict-free LDS.128
        const uint4* p = reinterpret_cast<const uint4*>(stages + (size_t)(s % (uint32_t)K) * SUB * 32) +
                         2 * (tid % SUB);
        const int h = (lane >> 2) & 1;
        const uint4 a = p[h], b = p[h ^ 1];
        const uint4 lo = h ? b : a, hi = h ? a : b;
        rank = lo.x; step = lo.y; sig = lo.z; phase = lo.w >> 16;
        start = (long long)(((unsigned long long)hi.y << 32) | hi.x);
        end = (long long)(((unsigned long long)hi.w << 32) | hi.z);
        pending = argus_event_key(D, rank, step, sig, phase, start, end, key);
        if (pending) ++n_valid; else ++n_invalid;
      }
    }
    bool ovf = false;
    for (;;) {
      const bool accept = pending && key == cur_key;
      // ---- spans: warp-uniform fast path in registers, else per-phase ballot groups -----------
      const uint32_t ph0 = __shfl_sync(FULL, phase, 0);
      if (__all_sync(FULL, accept && phase == ph0)) {
        if (ws.phase != ph0) { ws.flush(c.spans, lane); ws.phase = ph0; }
        ws.mn = start < ws.mn ? start : ws.mn;
        ws.mx = end > ws.mx ? end : ws.mx;
        ws.n++;
      } else {
        uint32_t todo = __ballot_sync(FULL, accept);
        while (todo) {
          const int leader = __ffs((int)todo) - 1;
          const uint32_t ph = __shfl_sync(FULL, phase, leader);
          const bool mine = accept && phase == ph;
          const uint32_t grp = __ballot_sync(FULL, mine);
          const long long a = warp_min_i64(mine ? start : INT64_MAX);
          const long long b = warp_max_i64(mine ? end : INT64_MIN);
          if (lane == leader) {
            atomicMin(&c.spans[ph].mn, a);
            atomicMax(&c.spans[ph].mx, b);
            atomicAdd(&c.spans[ph].n, (unsigned long long)__popc(grp));
          }
          todo &= ~grp;
        }
      }
      // ---- cells -----------------------------------------------------------------------------
      if (accept) {
        if (!cell_accumulate(c.table, sig, (uint64_t)(end - start))) {
          ovf = true;
          c.H->flags = 1u;
        }
        pending = false;
      }
      const int any_pending = __syncthreads_or(pending ? 1 : 0);
      if (c.H->flags) {  // uniform: written before the barrier
        // rare: some event does not fit the compact cell -> make the record live, then L2 atomics
        { ws.flush(c.spans, lane); flush_table(c, cur_key); }
        if (ovf) {
          // the span part was already folded above; only the cell goes the global way
          uint8_t* rec = records + (size_t)cur_key * D.rec_bytes;
          const uint64_t d = (uint64_t)(end - start);
          argus_cell* cl = reinterpret_cast<argus_cell*>(rec + D.cell_off) + sig;
          atomicAdd(reinterpret_cast<unsigned long long*>(&cl->count), 1ull);
          atomicAdd(reinterpret_cast<unsigned long long*>(&cl->sum_ns), (unsigned long long)d);
          atomicMin(reinterpret_cast<unsigned long long*>(&cl->min_ns), (unsigned long long)d);
          atomicMax(reinterpret_cast<unsigned long long*>(&cl->max_ns), (unsigned long long)d);
          atomicAdd(&cl->hist[argus_bucket64(d)], 1u);
          ovf = false;
        }
        if (tid == 0) c.H->flags = 0u;
        __syncthreads();
      }
      if (!any_pending) break;
      // ---- key switch: flush the finished record, adopt the key of the first pending event -----
      if (cur_key != KEY_NONE) { ws.flush(c.spans, lane); flush_table(c, cur_key); }
      if (pending) atomicMin(&c.H->next_idx, (uint32_t)tid);
      __syncthreads();
      if ((uint32_t)tid == c.H->next_idx) c.H->cur_key = key;
      __syncthreads();
      cur_key = c.H->cur_key;
      if (tid == 0) c.H->next_idx = KEY_NONE;
      // (next_idx is next read after at least one more barrier)
    }
    // every thread is past its reads of this iteration's stages: refill them
    if (tid == 0) {
      for (uint32_t g = 0; g < (uint32_t)G; ++g) {
        const uint32_t sn = it * G + (uint32_t)K + g;
        if (sn < n_sub) issue(sn);
      }
    }
  }
  if (cur_key != KEY_NONE) { ws.flush(c.spans, lane); flush_table(c, cur_key); }

  n_valid = __reduce_add_sync(FULL, n_valid);
  n_invalid = __reduce_add_sync(FULL, n_invalid);
  if (lane == 0) {
    if (n_valid) atomicAdd(&counters[0], (unsigned long long)n_valid);
    if (n_invalid) atomicAdd(&counters[1], (unsigned long long)n_invalid);
  }
}

size_t seg_fixed_smem(uint32_t S) { return (HDR_BYTES + SPAN_BYTES + 32u * (size_t)S + 127u) & ~(size_t)127u; }

}  // namespace

bool argus_seg_supported(const argus_ctx* ctx) {
  return seg_fixed_smem(ctx->dims.S) + (size_t)(G + 1) * SUB * 32 <= (size_t)ctx->max_smem_optin;
}

cudaError_t argus_launch_aggregate_seg(argus_ctx* ctx, const argus_event* ev, uint64_t n,
                                       void* d_records, cudaStream_t s) {
  if (n == 0) return cudaSuccess;
  const size_t fixed = seg_fixed_smem(ctx->dims.S);
  int K = (int)(((size_t)ctx->max_smem_optin - fixed) / ((size_t)SUB * 32));
  if (K > MAXK) K = MAXK;
  const size_t smem = fixed + (size_t)K * SUB * 32;
  cudaError_t e = cudaFuncSetAttribute(aggregate_seg_kernel,
                                       cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
  if (e != cudaSuccess) return e;
  int grid = ctx->tune_grid > 0 ? ctx->tune_grid : ctx->sm_count;
  // a CTA's slot counters hold 26 bits between flushes: bound the span of one CTA
  const uint64_t cap = (1ull << 26) - NT;
  uint64_t per_cta = (n + grid - 1) / grid;
  if (per_cta > cap) per_cta = cap;
  per_cta = (per_cta + NT - 1) / NT * NT;
  const uint64_t ctas = (n + per_cta - 1) / per_cta;
  aggregate_seg_kernel<<<(unsigned)ctas, NT, smem, s>>>(
      reinterpret_cast<const uint4*>(ev), n, per_cta, static_cast<uint8_t*>(d_records), ctx->d_state,
      ctx->d_counters, ctx->dims, K);
  return cudaGetLastError();
}
