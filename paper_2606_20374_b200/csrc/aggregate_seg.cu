// aggregate_seg.cu — segmented aggregation kernel (NS (3): "hand-written sm_100a aggregation
// kernels ... coalesced 128-bit vectorised loads, with TMA ... staging into shared memory ...
// shared-memory-privatised per-block histograms and min/max/sum ... warp-shuffle segmented
// reductions where a block spans rank-step boundaries, and flush to global in one pass").
//
// One persistent CTA per SM walks a contiguous span of the event buffer.  Events arrive through a
// ring of 8 KB stages filled by 1-D TMA bulk copies (cp.async.bulk + mbarrier complete_tx, L2
// evict-first).  Each thread takes EPT events per iteration into registers; the stages are
// refilled right after that load phase, so the whole ring is in flight while the CTA accumulates.
// The CTA keeps ONE (rank, step) table in shared memory at a time, 32 bytes per sig, laid out as
// structure-of-arrays so that random sigs spread over all 32 banks:
//   slots[S]  uint4: four tagged histogram slots {bucket+1 : 6 bits | count : 26 bits}; the word
//                    a slot lives in is XOR-swizzled with sig bits 3-4
//   sum_lo[S], sum_hi[S] u32: the 64-bit sum with an explicit carry
//   mm[S]     uint2: {~min, max} as u32
// Only native 32-bit shared atomics are used (64-bit shared atomics are CAS loops on sm_100a).
// An event the compact cell cannot take (duration >= 2^32 ns, or a fifth distinct bucket of one
// sig) goes straight to the global record with L2 atomics.  When the (rank, step) key changes the
// table is flushed: the first CTA to reach a record claims it and writes the whole 160-byte cells
// with coalesced 128-bit stores (no read-modify-write, no separate identity fill); any later
// contribution to the same record merges with L2 reductions.  Correct for ANY event order; fast
// when events are grouped by (rank, step) (R18).
#include "argus_internal.cuh"

namespace {

constexpr int SUB = 256;             // events per TMA stage (8 KB)
constexpr int MAXK = 24;             // ring stages (bounded by shared memory at launch)
constexpr uint32_t KEY_NONE = 0xFFFFFFFFu;
constexpr uint32_t FULL = 0xFFFFFFFFu;
constexpr uint32_t HDR_BYTES = 256;
constexpr uint32_t SPAN_BYTES = ARGUS_MAX_PHASES * 32;
constexpr uint32_t TAB_OFF = HDR_BYTES + SPAN_BYTES;   // compact table starts here

struct SpanAcc {                      // shared-memory span accumulator of one phase (32 B)
  long long mn, mx;
  unsigned long long n;
  unsigned long long pad;
};

struct Hdr {
  unsigned long long bars[MAXK];      // mbarriers, one per stage
  uint32_t cur_key;
  uint32_t flags;                     // != 0: some event of this iteration needs the global path
  uint32_t next_idx;                  // lowest pending event index (key switch)
  uint32_t mode;                      // state word seen by the flush claim
};
static_assert(sizeof(Hdr) <= HDR_BYTES, "header");

extern __shared__ __align__(128) uint8_t smem[];

// The compact table of one (rank, step), addressed by 32-bit offsets from the dynamic shared
// window: slots[S] uint4 | sum_lo[S] u32 | sum_hi[S] u32 | mm[S] uint2 {~min, max}.
struct Table {
  uint32_t S;
  __device__ __forceinline__ uint4* slots(uint32_t sig) const { return reinterpret_cast<uint4*>(smem + TAB_OFF) + sig; }
  __device__ __forceinline__ uint32_t* slot_words(uint32_t sig) const { return reinterpret_cast<uint32_t*>(smem + TAB_OFF) + 4u * sig; }
  __device__ __forceinline__ uint32_t* sum_lo(uint32_t sig) const { return reinterpret_cast<uint32_t*>(smem + TAB_OFF + 16u * S) + sig; }
  __device__ __forceinline__ uint32_t* sum_hi(uint32_t sig) const { return reinterpret_cast<uint32_t*>(smem + TAB_OFF + 20u * S) + sig; }
  __device__ __forceinline__ uint2* mm(uint32_t sig) const { return reinterpret_cast<uint2*>(smem + TAB_OFF + 24u * S) + sig; }
};
__device__ __forceinline__ Hdr* hdr() { return reinterpret_cast<Hdr*>(smem); }
__device__ __forceinline__ SpanAcc* span_tab() { return reinterpret_cast<SpanAcc*>(smem + HDR_BYTES); }
__host__ __device__ __forceinline__ uint32_t stage_off(uint32_t S) {
  return (TAB_OFF + 32u * ((S + 3u) & ~3u) + 127u) & ~127u;
}

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
                                            uint32_t bar, uint64_t policy) {
  asm volatile(
      "cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes.L2::cache_hint "
      "[%0], [%1], %2, [%3], %4;" ::"r"(dst),
      "l"(src), "r"(bytes), "r"(bar), "l"(policy)
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
  __device__ __forceinline__ void flush(int lane) {
    if (phase != KEY_NONE) {
      long long a = warp_min_i64(mn), b = warp_max_i64(mx);
      uint32_t c = __reduce_add_sync(FULL, n);
      if (lane == 0 && c) {
        SpanAcc* sp = span_tab() + phase;
        atomicMin(&sp->mn, a);
        atomicMax(&sp->mx, b);
        atomicAdd(&sp->n, (unsigned long long)c);
      }
    }
    reset();
  }
};

struct Glob {             // global-memory side of the kernel
  uint8_t* records;
  uint32_t* state;
  argus_dims D;
};

// Histogram part of one event: bump the slot tagged bucket+1, claiming one if needed.
// `s` is a (possibly stale) snapshot of the sig's four slot words.  Returns false if all four
// slots hold other buckets.
__device__ __forceinline__ bool slot_update(const Table& tb, uint32_t sig, uint32_t tag, const uint4& s) {
  uint32_t* w = tb.slot_words(sig);
  int p = -1;
  if ((s.x & 63u) == tag) p = 0;
  else if ((s.y & 63u) == tag) p = 1;
  else if ((s.z & 63u) == tag) p = 2;
  else if ((s.w & 63u) == tag) p = 3;
  if (p >= 0) {
    atomicAdd(w + p, 64u);
    return true;
  }
  // claim (first events of a bucket in this rank-step).  Slots are claimed in a fixed per-sig
  // order (logical j -> word j ^ swz) and never released before the flush, so a tag lives in at
  // most one slot.  The swizzle spreads the first-claimed (hottest) slot over all banks.
  const int swz = (int)((sig >> 3) & 3u);
#pragma unroll 1
  for (int j = 0; j < 4; ++j) {
    uint32_t* q = w + (j ^ swz);
    uint32_t v = *reinterpret_cast<volatile uint32_t*>(q);
    if (v == 0u) {
      v = atomicCAS(q, 0u, tag | 64u);
      if (v == 0u) return true;
    }
    if ((v & 63u) == tag) { atomicAdd(q, 64u); return true; }
  }
  return false;
}

// 16-byte chunk `part` (0..9) of the 160-byte argus_cell decoded from a compact cell.
__device__ __forceinline__ uint4 cell_chunk(const uint4 s, uint32_t sum_lo, uint32_t sum_hi,
                                            const uint2 m, uint32_t part) {
  const uint32_t c0 = s.x >> 6, c1 = s.y >> 6, c2 = s.z >> 6, c3 = s.w >> 6;
  if (part == 0u) {
    unsigned long long cnt = (unsigned long long)c0 + c1 + c2 + c3;
    return make_uint4((uint32_t)cnt, (uint32_t)(cnt >> 32), sum_lo, sum_hi);
  }
  if (part == 1u) {
    if ((c0 | c1 | c2 | c3) == 0u) return make_uint4(0xFFFFFFFFu, 0xFFFFFFFFu, 0u, 0u);
    return make_uint4(~m.x, 0u, m.y, 0u);
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

// Flush the shared table of record `key` to global memory and clear it.  All threads call; the
// caller has flushed its WarpSpan first.
template <int NT>
__device__ __noinline__ void flush_table(const Glob& g, uint32_t key) {
  const int tid = threadIdx.x;
  const argus_dims& D = g.D;
  const Table tb{D.S};
  Hdr* H = hdr();
  SpanAcc* spans = span_tab();
  __syncthreads();
  if (tid == 0) {
    uint32_t old = atomicCAS(&g.state[key], ARGUS_ST_LAZY, ARGUS_ST_BUSY);
    if (old == ARGUS_ST_BUSY) {
      // another (resident, running) CTA is writing this record: wait for it, then merge
      while (atomicAdd(&g.state[key], 0u) != ARGUS_ST_LIVE) __nanosleep(128);
      __threadfence();
      old = ARGUS_ST_LIVE;
    }
    H->mode = old;
  }
  __syncthreads();
  const uint32_t mode = H->mode;
  uint8_t* rec = g.records + (size_t)key * D.rec_bytes;
  if (mode == ARGUS_ST_LAZY) {
    // we own the record: write spans + cells once, coalesced 16-byte chunks
    uint4* dst = reinterpret_cast<uint4*>(rec + D.span_off);
    const uint32_t span_chunks = 2u * (D.P + 1u);
    const uint32_t n_chunks = span_chunks + 10u * D.S;
    for (uint32_t ch = tid; ch < n_chunks; ch += NT) {
      uint4 v;
      if (ch < span_chunks) {
        const uint32_t k = ch >> 1;
        if (k < D.P && spans[k].n != 0ull) {
          const SpanAcc a = spans[k];
          v = (ch & 1u) ? make_uint4(0u, 0u, (uint32_t)a.n, (uint32_t)(a.n >> 32))
                        : make_uint4((uint32_t)a.mn, (uint32_t)((unsigned long long)a.mn >> 32),
                                     (uint32_t)a.mx, (uint32_t)((unsigned long long)a.mx >> 32));
        } else {
          v = argus_identity_chunk(D, ch);
        }
      } else {
        const uint32_t cc = ch - span_chunks;
        const uint32_t sig = cc / 10u, part = cc - sig * 10u;
        v = cell_chunk(*tb.slots(sig), *tb.sum_lo(sig), *tb.sum_hi(sig), *tb.mm(sig), part);
      }
      __stcs(dst + ch, v);
    }
    __threadfence();
    __syncthreads();
    if (tid == 0) atomicExch(&g.state[key], ARGUS_ST_LIVE);
  } else {
    // merge into a live record with L2 reductions (non-empty fields only)
    argus_cell* cells = reinterpret_cast<argus_cell*>(rec + D.cell_off);
    for (uint32_t sig = tid; sig < D.S; sig += NT) {
      const uint4 s = *tb.slots(sig);
      const uint2 m = *tb.mm(sig);
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
                  ((unsigned long long)*tb.sum_hi(sig) << 32) | *tb.sum_lo(sig));
        atomicMin(reinterpret_cast<unsigned long long*>(&cells[sig].min_ns),
                  (unsigned long long)(~m.x));
        atomicMax(reinterpret_cast<unsigned long long*>(&cells[sig].max_ns),
                  (unsigned long long)m.y);
      }
    }
    argus_span* sp = reinterpret_cast<argus_span*>(rec + D.span_off);
    for (uint32_t k = tid; k < D.P; k += NT) {
      const SpanAcc a = spans[k];
      if (a.n) {
        atomicMin(reinterpret_cast<long long*>(&sp[k].min_start_ns), a.mn);
        atomicMax(reinterpret_cast<long long*>(&sp[k].max_end_ns), a.mx);
        atomicAdd(reinterpret_cast<unsigned long long*>(&sp[k].n_events), a.n);
      }
    }
  }
  __syncthreads();
  uint4* all = tb.slots(0);           // slots, sum_lo, sum_hi, mm are contiguous: 2*S uint4
  for (uint32_t i = tid; i < 2u * D.S; i += NT) all[i] = make_uint4(0u, 0u, 0u, 0u);
  for (uint32_t k = tid; k < D.P; k += NT) {
    spans[k].mn = INT64_MAX; spans[k].mx = INT64_MIN; spans[k].n = 0ull; spans[k].pad = 0ull;
  }
  __syncthreads();
}

template <int NT, int EPT>
__global__ void __launch_bounds__(NT, 1)
aggregate_seg_kernel(const uint4* __restrict__ ev, uint64_t n, uint64_t per_cta, uint8_t* records,
                     uint32_t* state, unsigned long long* counters, argus_dims D, int K) {
  constexpr int G = EPT * NT / SUB;    // stages consumed per iteration
  constexpr int WPS = NT / SUB;        // stage groups per event slot (threads / stage size)
  static_assert(NT % SUB == 0 && G >= 1, "geometry");
  Glob gl;
  gl.records = records; gl.state = state; gl.D = D;
  const Table tb{D.S};
  Hdr* H = hdr();
  const uint32_t stages = stage_off(D.S);     // byte offset of the stage ring in smem

  const int tid = threadIdx.x, lane = tid & 31;
  const uint64_t e0 = (uint64_t)blockIdx.x * per_cta;
  if (e0 >= n) return;
  const uint64_t e1 = (e0 + per_cta < n) ? e0 + per_cta : n;
  const uint32_t n_ev = (uint32_t)(e1 - e0);
  const uint32_t n_sub = (n_ev + SUB - 1) / SUB;
  const uint32_t n_iter = (n_ev + EPT * NT - 1) / (EPT * NT);
  const uint4* src = ev + 2 * e0;

  if (tid == 0) {
    for (int k = 0; k < K; ++k) mbar_init(smem_u32(&H->bars[k]), 1u);
    H->cur_key = KEY_NONE; H->flags = 0u; H->next_idx = KEY_NONE; H->mode = 0u;
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
  }
  {
    uint4* all = tb.slots(0);
    for (uint32_t i = tid; i < 2u * D.S; i += NT) all[i] = make_uint4(0u, 0u, 0u, 0u);
    SpanAcc* spans = span_tab();
    for (uint32_t k = tid; k < ARGUS_MAX_PHASES; k += NT) {
      spans[k].mn = INT64_MAX; spans[k].mx = INT64_MIN; spans[k].n = 0ull; spans[k].pad = 0ull;
    }
  }
  __syncthreads();

  uint64_t policy = 0;
  if (tid == 0) asm volatile("createpolicy.fractional.L2::evict_first.b64 %0, 1.0;" : "=l"(policy));
  auto issue = [&](uint32_t s, uint32_t slot) {  // thread 0 only: stage s into ring slot `slot`
    const uint32_t cnt = (n_ev - s * SUB < (uint32_t)SUB) ? n_ev - s * SUB : (uint32_t)SUB;
    const uint32_t bar = smem_u32(&H->bars[slot]);
    mbar_expect_tx(bar, cnt * 32u);
    tma_load_1d(smem_u32(smem + stages + slot * (SUB * 32u)), src + 2 * (size_t)s * SUB, cnt * 32u, bar, policy);
  };
  if (tid == 0)
    for (uint32_t s = 0; s < (uint32_t)K && s < n_sub; ++s) issue(s, s);

  WarpSpan ws;
  ws.reset();
  uint32_t cur_key = KEY_NONE;
  uint32_t n_invalid = 0;
  // ring position of stage it*G + tid/SUB (this thread's first stage); the others follow at +WPS
  uint32_t slot0 = (uint32_t)(tid / SUB) % (uint32_t)K, par0 = 0;
  uint32_t base_slot = 0;

  for (uint32_t it = 0; it < n_iter; ++it) {
    // ---- load phase: EPT events per thread, stage -> registers ---------------------------------
    uint32_t sig[EPT], phase[EPT], key[EPT];
    long long start[EPT], end[EPT];
    bool pending[EPT];
    {
      uint32_t sl = slot0, pr = par0;
#pragma unroll
      for (int e = 0; e < EPT; ++e) {
        const uint32_t s = it * G + (uint32_t)(e * WPS + tid / SUB);
        const uint32_t idx = it * (EPT * NT) + (uint32_t)(e * NT + tid);
        pending[e] = false; sig[e] = 0; phase[e] = 0; key[e] = KEY_NONE; start[e] = 0; end[e] = 0;
        if (s < n_sub) {
          mbar_wait(smem_u32(&H->bars[sl]), pr);
          if (idx < n_ev) {
            // lanes 0-3,8-11,.. read the first half first, the others the second: conflict-free LDS.128
            const uint4* p = reinterpret_cast<const uint4*>(smem + stages + sl * (SUB * 32u)) + 2 * (tid % SUB);
            const int h = (lane >> 2) & 1;
            const uint4 a = p[h], b = p[h ^ 1];
            const uint4 lo = h ? b : a, hi = h ? a : b;
            sig[e] = lo.z; phase[e] = lo.w >> 16;
            start[e] = (long long)(((unsigned long long)hi.y << 32) | hi.x);
            end[e] = (long long)(((unsigned long long)hi.w << 32) | hi.z);
            pending[e] = argus_event_key(D, lo.x, lo.y, lo.z, phase[e], start[e], end[e], key[e]);
            n_invalid += pending[e] ? 0u : 1u;
          }
        }
        sl += WPS; if (sl >= (uint32_t)K) { sl -= (uint32_t)K; pr ^= 1u; }
      }
      slot0 = sl; par0 = pr;     // EPT*WPS = G stages further
    }
    __syncthreads();   // every thread holds its events: the G stages can be refilled right away
    if (tid == 0) {
      uint32_t sl = base_slot;
#pragma unroll 1
      for (uint32_t g = 0; g < (uint32_t)G; ++g) {
        const uint32_t sn = it * G + (uint32_t)K + g;
        if (sn < n_sub) issue(sn, sl);
        if (++sl == (uint32_t)K) sl = 0;
      }
    }
    base_slot += G; if (base_slot >= (uint32_t)K) base_slot -= (uint32_t)K;

    uint32_t ovf_mask = 0;
    for (;;) {
      bool accept[EPT];
      uint4 snap[EPT];
      uint2 mmv[EPT];
      // ---- table loads for all accepted events first (ILP), then the atomics ---------------------
#pragma unroll
      for (int e = 0; e < EPT; ++e) {
        accept[e] = pending[e] && key[e] == cur_key;
        if (accept[e]) { snap[e] = *tb.slots(sig[e]); mmv[e] = *tb.mm(sig[e]); }
      }
      // ---- spans: warp-uniform fast path in registers, else per-phase ballot groups ---------------
#pragma unroll
      for (int e = 0; e < EPT; ++e) {
        const uint32_t ph0 = __shfl_sync(FULL, phase[e], 0);
        if (__all_sync(FULL, accept[e] && phase[e] == ph0)) {
          if (ws.phase != ph0) { ws.flush(lane); ws.phase = ph0; }
          ws.mn = start[e] < ws.mn ? start[e] : ws.mn;
          ws.mx = end[e] > ws.mx ? end[e] : ws.mx;
          ws.n++;
        } else {
          uint32_t todo = __ballot_sync(FULL, accept[e]);
          while (todo) {
            const int leader = __ffs((int)todo) - 1;
            const uint32_t ph = __shfl_sync(FULL, phase[e], leader);
            const bool mine = accept[e] && phase[e] == ph;
            const uint32_t grp = __ballot_sync(FULL, mine);
            const long long a = warp_min_i64(mine ? start[e] : INT64_MAX);
            const long long b = warp_max_i64(mine ? end[e] : INT64_MIN);
            if (lane == leader) {
              SpanAcc* sp = span_tab() + ph;
              atomicMin(&sp->mn, a);
              atomicMax(&sp->mx, b);
              atomicAdd(&sp->n, (unsigned long long)__popc(grp));
            }
            todo &= ~grp;
          }
        }
      }
      // ---- cells ------------------------------------------------------------------------------------
      uint32_t d32[EPT], old[EPT];
      bool fits[EPT];
#pragma unroll
      for (int e = 0; e < EPT; ++e) {
        const unsigned long long d = (unsigned long long)(end[e] - start[e]);
        d32[e] = (uint32_t)d;
        fits[e] = accept[e] && (d >> 32) == 0ull;
        if (fits[e]) {
          const uint32_t tag = (31u - (uint32_t)__clz((int)(d32[e] | 1u))) + 1u;  // bucket + 1
          fits[e] = slot_update(tb, sig[e], tag, snap[e]);
        }
        if (accept[e] && !fits[e]) { ovf_mask |= 1u << e; H->flags = 1u; }
      }
#pragma unroll
      for (int e = 0; e < EPT; ++e)
        if (fits[e]) old[e] = atomicAdd(tb.sum_lo(sig[e]), d32[e]);
#pragma unroll
      for (int e = 0; e < EPT; ++e)
        if (fits[e]) {
          if (~d32[e] > mmv[e].x) atomicMax(&tb.mm(sig[e])->x, ~d32[e]);
          if (d32[e] > mmv[e].y) atomicMax(&tb.mm(sig[e])->y, d32[e]);
        }
      bool pend = false;
#pragma unroll
      for (int e = 0; e < EPT; ++e) {
        if (fits[e] && old[e] + d32[e] < old[e]) atomicAdd(tb.sum_hi(sig[e]), 1u);
        if (accept[e]) pending[e] = false;
        pend |= pending[e];
      }
      const int any_pending = __syncthreads_or(pend ? 1 : 0);
      if (H->flags) {  // uniform: written before the barrier
        // rare: some event does not fit the compact cell -> make the record live, then L2 atomics
        ws.flush(lane);
        flush_table<NT>(gl, cur_key);
#pragma unroll
        for (int e = 0; e < EPT; ++e)
          if (ovf_mask & (1u << e)) {
            // the span part was already folded above; only the cell goes the global way
            uint8_t* rec = records + (size_t)cur_key * D.rec_bytes;
            const uint64_t d = (uint64_t)(end[e] - start[e]);
            argus_cell* cl = reinterpret_cast<argus_cell*>(rec + D.cell_off) + sig[e];
            atomicAdd(reinterpret_cast<unsigned long long*>(&cl->count), 1ull);
            atomicAdd(reinterpret_cast<unsigned long long*>(&cl->sum_ns), (unsigned long long)d);
            atomicMin(reinterpret_cast<unsigned long long*>(&cl->min_ns), (unsigned long long)d);
            atomicMax(reinterpret_cast<unsigned long long*>(&cl->max_ns), (unsigned long long)d);
            atomicAdd(&cl->hist[argus_bucket64(d)], 1u);
          }
        ovf_mask = 0;
        if (tid == 0) H->flags = 0u;
        __syncthreads();
      }
      if (!any_pending) break;
      // ---- key switch: flush the finished record, adopt the key of the first pending event --------
      if (cur_key != KEY_NONE) { ws.flush(lane); flush_table<NT>(gl, cur_key); }
#pragma unroll
      for (int e = EPT - 1; e >= 0; --e)
        if (pending[e]) atomicMin(&H->next_idx, (uint32_t)(e * NT + tid));
      __syncthreads();
      {
        const uint32_t pick = H->next_idx;
#pragma unroll
        for (int e = 0; e < EPT; ++e)
          if ((uint32_t)(e * NT + tid) == pick) H->cur_key = key[e];
      }
      __syncthreads();
      cur_key = H->cur_key;
      if (tid == 0) H->next_idx = KEY_NONE;
      // (next_idx is next read after at least one more barrier)
    }
  }
  if (cur_key != KEY_NONE) { ws.flush(lane); flush_table<NT>(gl, cur_key); }

  n_invalid = __reduce_add_sync(FULL, n_invalid);
  if (lane == 0 && n_invalid) atomicAdd(&counters[1], (unsigned long long)n_invalid);
  if (tid == 0) atomicAdd(&counters[0], (unsigned long long)n_ev);   // valid = seen - invalid (host)
}

template <int NT, int EPT>
cudaError_t launch_variant(argus_ctx* ctx, const argus_event* ev, uint64_t n, void* d_records,
                           cudaStream_t s) {
  constexpr int G = EPT * NT / SUB;
  const size_t fixed = stage_off(ctx->dims.S);
  int K = (int)(((size_t)ctx->max_smem_optin - fixed) / ((size_t)SUB * 32));
  if (K > MAXK) K = MAXK;
  if (K < G) return cudaErrorInvalidConfiguration;
  const size_t smem_bytes = fixed + (size_t)K * SUB * 32;
  cudaError_t e = cudaFuncSetAttribute(aggregate_seg_kernel<NT, EPT>,
                                       cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem_bytes);
  if (e != cudaSuccess) return e;
  int grid = ctx->tune_grid > 0 ? ctx->tune_grid : ctx->sm_count;
  // a CTA's slot counters hold 26 bits between flushes: bound the span of one CTA
  const uint64_t tile = (uint64_t)EPT * NT;
  const uint64_t cap = (1ull << 26) - tile;
  uint64_t per_cta = (n + grid - 1) / grid;
  if (per_cta > cap) per_cta = cap;
  per_cta = (per_cta + tile - 1) / tile * tile;
  const uint64_t ctas = (n + per_cta - 1) / per_cta;
  aggregate_seg_kernel<NT, EPT><<<(unsigned)ctas, NT, smem_bytes, s>>>(
      reinterpret_cast<const uint4*>(ev), n, per_cta, static_cast<uint8_t*>(d_records), ctx->d_state,
      ctx->d_counters, ctx->dims, K);
  return cudaGetLastError();
}

}  // namespace

bool argus_seg_supported(const argus_ctx* ctx) {
  // the smallest variant consumes 4 stages (32 KB) per iteration
  return (size_t)stage_off(ctx->dims.S) + (size_t)8 * SUB * 32 <= (size_t)ctx->max_smem_optin;
}

cudaError_t argus_launch_aggregate_seg(argus_ctx* ctx, const argus_event* ev, uint64_t n,
                                       void* d_records, cudaStream_t s) {
  if (n == 0) return cudaSuccess;
  switch (ctx->tune_variant) {
    case 1: return launch_variant<1024, 1>(ctx, ev, n, d_records, s);
    case 2: return launch_variant<1024, 2>(ctx, ev, n, d_records, s);
    case 3: return launch_variant<512, 2>(ctx, ev, n, d_records, s);
    case 5: return launch_variant<256, 8>(ctx, ev, n, d_records, s);
    case 6: return launch_variant<768, 2>(ctx, ev, n, d_records, s);
    case 4:
    default: return launch_variant<512, 4>(ctx, ev, n, d_records, s);
  }
}
