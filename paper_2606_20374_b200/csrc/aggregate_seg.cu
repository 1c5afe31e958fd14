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

constexpr int MAXK = 48;             // ring stages (bounded by shared memory at launch)
constexpr uint32_t KEY_NONE = 0xFFFFFFFFu;
constexpr uint32_t FULL = 0xFFFFFFFFu;
constexpr uint32_t HDR_BYTES = 1024;
constexpr uint32_t SPAN_BYTES = ARGUS_MAX_PHASES * 32;
constexpr uint32_t TAB_OFF = HDR_BYTES + SPAN_BYTES;   // compact table starts here

struct SpanAcc {                      // shared-memory span accumulator of one phase (32 B)
  long long mn, mx;
  unsigned long long n;
  unsigned long long pad;
};

struct Hdr {
  unsigned long long full[MAXK];      // mbarriers: stage filled by TMA (tx bytes)
  unsigned long long empty[MAXK];     // mbarriers: stage read by all its consumer warps
  uint32_t cur_key;                   // key adopted at the rendezvous
  uint32_t pad0;
  uint32_t next_idx;                  // lowest pending event index
  uint32_t mode;                      // state word seen by the flush claim
  uint32_t n_finished;                // consumer warps that ran out of events
  uint32_t decision;                  // outcome of the current rendezvous
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

__device__ __forceinline__ bool mbar_try_wait(uint32_t bar, uint32_t parity) {
  uint32_t ok;
  asm volatile(
      "{\n"
      ".reg .pred P1;\n"
      "mbarrier.try_wait.parity.shared::cta.b64 P1, [%1], %2, %3;\n"
      "selp.u32 %0, 1, 0, P1;\n"
      "}"
      : "=r"(ok)
      : "r"(bar), "r"(parity), "r"(2000u)   // suspend-time hint (ns): fewer wasted polls while waiting
      : "memory");
  return ok != 0u;
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
      const uint32_t c = n;              // warp-uniform
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

__device__ __forceinline__ void bar_consumers(int n) {   // named barrier 1: consumer warps only
  asm volatile("bar.sync 1, %0;" ::"r"(n) : "memory");
}
__device__ __forceinline__ void mbar_arrive(uint32_t bar) {
  asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(bar) : "memory");
}

// Flush the shared table of record `key` to global memory and clear it.  All NC consumer threads
// call (tid < NC); each warp has flushed its WarpSpan first.  Ends with a consumer barrier.
template <int NC>
__device__ __noinline__ void flush_table(const Glob& g, uint32_t key) {
  const int tid = threadIdx.x;
  const argus_dims& D = g.D;
  const Table tb{D.S};
  Hdr* H = hdr();
  SpanAcc* spans = span_tab();
  bar_consumers(NC);
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
  bar_consumers(NC);
  const uint32_t mode = H->mode;
  uint8_t* rec = g.records + (size_t)key * D.rec_bytes;
  if (mode == ARGUS_ST_LAZY) {
    // we own the record: write spans + cells once, coalesced 16-byte chunks
    uint4* dst = reinterpret_cast<uint4*>(rec + D.span_off);
    const uint32_t span_chunks = 2u * (D.P + 1u);
    const uint32_t n_chunks = span_chunks + 10u * D.S;
    for (uint32_t ch = tid; ch < n_chunks; ch += NC) {
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
    bar_consumers(NC);
    if (tid == 0) atomicExch(&g.state[key], ARGUS_ST_LIVE);
  } else {
    // merge into a live record with L2 reductions (non-empty fields only)
    argus_cell* cells = reinterpret_cast<argus_cell*>(rec + D.cell_off);
    for (uint32_t sig = tid; sig < D.S; sig += NC) {
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
    for (uint32_t k = tid; k < D.P; k += NC) {
      const SpanAcc a = spans[k];
      if (a.n) {
        atomicMin(reinterpret_cast<long long*>(&sp[k].min_start_ns), a.mn);
        atomicMax(reinterpret_cast<long long*>(&sp[k].max_end_ns), a.mx);
        atomicAdd(reinterpret_cast<unsigned long long*>(&sp[k].n_events), a.n);
      }
    }
  }
  bar_consumers(NC);
  uint4* all = tb.slots(0);           // slots, sum_lo, sum_hi, mm are contiguous: 2*S uint4
  for (uint32_t i = tid; i < 2u * D.S; i += NC) all[i] = make_uint4(0u, 0u, 0u, 0u);
  for (uint32_t k = tid; k < D.P; k += NC) {
    spans[k].mn = INT64_MAX; spans[k].mx = INT64_MIN; spans[k].n = 0ull; spans[k].pad = 0ull;
  }
  bar_consumers(NC);
}

// Rendezvous of all consumer warps (the only CTA-wide synchronisation of the steady state, taken
// once per (rank, step) boundary on grouped input).  A warp comes here when it holds an event it
// cannot fold: another key than the table's, or an event that needs the global path while the
// record is not live yet.  Warps that see H->park_flag, or have run out of events, join.  Then the
// table is flushed and the key of the lowest pending event becomes current.  Returns true when no
// warp has anything left (the last table has been flushed).
// Result packed as {cur_key : 32 | live : 1 | all_done : 1} (by value: keeps the caller's state in registers).
constexpr unsigned long long PARK_LIVE = 1ull << 32, PARK_DONE = 1ull << 33;
constexpr uint32_t DEC_SWITCH = 0u, DEC_SPURIOUS = 1u, DEC_DONE = 2u;
template <int NC>
__device__ __noinline__ unsigned long long park(const Glob& gl, bool pending, uint32_t key,
                                                uint32_t my_idx, uint32_t cur_key, uint32_t live) {
  Hdr* H = hdr();
  const int tid = threadIdx.x;
  // a pending event's index is the rendezvous request: every warp whose position in the stream is
  // beyond H->next_idx comes here instead of going on (finished warps just wait here)
  if (pending) atomicMin(&H->next_idx, my_idx);
  bar_consumers(NC);
  const uint32_t pick = *reinterpret_cast<volatile uint32_t*>(&H->next_idx);
  if (tid == 0) {
    const uint32_t fin = *reinterpret_cast<volatile uint32_t*>(&H->n_finished);
    H->decision = pick != KEY_NONE ? DEC_SWITCH : (fin == (uint32_t)(NC / 32) ? DEC_DONE : DEC_SPURIOUS);
  }
  if (pending && my_idx == pick) H->cur_key = key;
  bar_consumers(NC);
  const uint32_t dec = *reinterpret_cast<volatile uint32_t*>(&H->decision);
  const uint32_t nk = *reinterpret_cast<volatile uint32_t*>(&H->cur_key);
  if (dec == DEC_SPURIOUS) {            // nobody holds a pending event, but not every warp is done
    bar_consumers(NC);
    return (unsigned long long)cur_key | (live ? PARK_LIVE : 0ull);
  }
  if (dec == DEC_DONE) {
    if (cur_key != KEY_NONE) flush_table<NC>(gl, cur_key);
    return PARK_DONE | cur_key;
  }
  if (cur_key != KEY_NONE) flush_table<NC>(gl, cur_key);   // begins and ends with a consumer barrier
  else bar_consumers(NC);
  if (tid == 0) H->next_idx = KEY_NONE;
  bar_consumers(NC);
  if (nk == cur_key) live = 1u;          // an overflow event asked for a live record
  else { cur_key = nk; live = 0u; }
  return (unsigned long long)cur_key | (live ? PARK_LIVE : 0ull);
}

// CW consumer warps + 1 producer warp.  Stage = WPSTG warps' worth of events (WPSTG KB).
template <int CW, int WPSTG>
__global__ void __launch_bounds__((CW + 1) * 32, 1)
aggregate_seg_kernel(const uint4* __restrict__ ev, uint64_t n, uint64_t per_cta, uint8_t* records,
                     uint32_t* state, unsigned long long* counters, argus_dims D, int K) {
  constexpr int NC = CW * 32;            // consumer threads
  constexpr int SUBE = WPSTG * 32;       // events per stage
  constexpr int SPI = CW / WPSTG;        // stages per iteration
  static_assert(CW % WPSTG == 0, "geometry");
  Glob gl;
  gl.records = records; gl.state = state; gl.D = D;
  const Table tb{D.S};
  Hdr* H = hdr();
  const uint32_t stages = stage_off(D.S);     // byte offset of the stage ring in smem

  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  const uint64_t e0 = (uint64_t)blockIdx.x * per_cta;
  if (e0 >= n) return;
  const uint64_t e1 = (e0 + per_cta < n) ? e0 + per_cta : n;
  const uint32_t n_ev = (uint32_t)(e1 - e0);
  const uint32_t n_sub = (n_ev + SUBE - 1) / SUBE;
  const uint32_t n_iter = (n_ev + NC - 1) / NC;
  const uint4* src = ev + 2 * e0;

  if (tid == 0) {
    for (int k = 0; k < K; ++k) {
      mbar_init(smem_u32(&H->full[k]), 1u);
      mbar_init(smem_u32(&H->empty[k]), (uint32_t)WPSTG);
    }
    H->cur_key = KEY_NONE; H->pad0 = 0u; H->next_idx = KEY_NONE; H->mode = 0u;
    H->n_finished = 0u; H->decision = 0u;
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
  }
  {
    uint4* all = tb.slots(0);
    for (uint32_t i = tid; i < 2u * D.S; i += (CW + 1) * 32) all[i] = make_uint4(0u, 0u, 0u, 0u);
    SpanAcc* spans = span_tab();
    for (uint32_t k = tid; k < ARGUS_MAX_PHASES; k += (CW + 1) * 32) {
      spans[k].mn = INT64_MAX; spans[k].mx = INT64_MIN; spans[k].n = 0ull; spans[k].pad = 0ull;
    }
  }
  __syncthreads();

  if (warp == CW) {
    // ---- producer warp: one lane streams the CTA's span through the ring with TMA bulk copies ----
    if (lane == 0) {
      uint64_t policy;
      asm volatile("createpolicy.fractional.L2::evict_first.b64 %0, 1.0;" : "=l"(policy));
      uint32_t slot = 0, round = 0;
      for (uint32_t s = 0; s < n_sub; ++s) {
        if (round) mbar_wait(smem_u32(&H->empty[slot]), (round - 1u) & 1u);
        const uint32_t cnt = (n_ev - s * SUBE < (uint32_t)SUBE) ? n_ev - s * SUBE : (uint32_t)SUBE;
        const uint32_t bar = smem_u32(&H->full[slot]);
        mbar_expect_tx(bar, cnt * 32u);
        tma_load_1d(smem_u32(smem + stages + slot * (SUBE * 32u)), src + 2 * (size_t)s * SUBE,
                    cnt * 32u, bar, policy);
        if (++slot == (uint32_t)K) { slot = 0; ++round; }
      }
    }
    return;
  }

  // ---- consumer warps -----------------------------------------------------------------------------
  WarpSpan ws;
  ws.reset();
  uint32_t cur_key = KEY_NONE, live = 0u;
  uint32_t n_invalid = 0;
  const uint32_t grp = (uint32_t)warp / WPSTG, wis = (uint32_t)warp % WPSTG;   // stage group, warp in stage
  uint32_t slot = grp % (uint32_t)K, par = (grp / (uint32_t)K) & 1u;
  uint32_t s = grp;                              // this warp's stage of the current iteration
  uint32_t my_pos = (uint32_t)warp * 32u;        // first event of this warp's chunk

  for (uint32_t it = 0; it < n_iter; ++it) {
    const uint32_t idx = my_pos + (uint32_t)lane;
    // ---- load: one event per lane, stage -> registers; release the stage at once --------------------
    const bool have = s < n_sub;                 // this warp's stage exists (warp-uniform)
    uint32_t sig = 0, phase = 0, key = KEY_NONE;
    long long start = 0, end = 0;
    bool pending = false;
    // While a warp waits for data it watches the rendezvous request: a warp beyond the requested
    // position joins the rendezvous BEFORE taking its next chunk (a parked warp keeps its next
    // stage unreleased, which may stall the in-order producer, so nobody may wait for data while
    // others wait for him).  Warps before that position go on: their stages are always issued.
    while (have && !mbar_try_wait(smem_u32(&H->full[slot]), par)) {
      if (*reinterpret_cast<volatile uint32_t*>(&H->next_idx) < my_pos) {
        ws.flush(lane);
        const unsigned long long r = park<NC>(gl, false, KEY_NONE, KEY_NONE, cur_key, live);
        cur_key = (uint32_t)r; live = (uint32_t)(r >> 32) & 1u;
      }
    }
    if (have) {
      if (idx < n_ev) {
        const uint4* p = reinterpret_cast<const uint4*>(smem + stages + slot * (SUBE * 32u)) + 2 * (wis * 32u + lane);
#if ARGUS_SEG_SWIZZLED_LOAD
        // lanes 0-3,8-11,.. read the first half first, the others the second: conflict-free LDS.128
        const int h = (lane >> 2) & 1;
        const uint4 a = p[h], b = p[h ^ 1];
        const uint4 lo = h ? b : a, hi = h ? a : b;
#else
        const uint4 lo = p[0], hi = p[1];
#endif
        sig = lo.z; phase = lo.w >> 16;
        start = (long long)(((unsigned long long)hi.y << 32) | hi.x);
        end = (long long)(((unsigned long long)hi.w << 32) | hi.z);
        pending = argus_event_key(D, lo.x, lo.y, lo.z, phase, start, end, key);
        n_invalid += pending ? 0u : 1u;
      }
      __syncwarp();
      if (lane == 0) mbar_arrive(smem_u32(&H->empty[slot]));
    }
    slot += SPI; if (slot >= (uint32_t)K) { slot -= (uint32_t)K; par ^= 1u; }
    s += SPI; my_pos += NC;

    for (;;) {
      // ---- cells -----------------------------------------------------------------------------------
      const bool accept = pending && key == cur_key;
      bool ok = false;
      if (accept) {
        const unsigned long long d = (unsigned long long)(end - start);
        const uint32_t d32 = (uint32_t)d;
        bool fits = (d >> 32) == 0ull;
        if (fits) {
          const uint32_t tag = (31u - (uint32_t)__clz((int)(d32 | 1u))) + 1u;  // bucket + 1
          const uint4 snap = *tb.slots(sig);
          const uint2 mmv = *tb.mm(sig);
          fits = slot_update(tb, sig, tag, snap);
          if (fits) {
            const uint32_t old = atomicAdd(tb.sum_lo(sig), d32);
            if ((~d32 > mmv.x) | (d32 > mmv.y)) {   // a new extreme: rare once a cell has a few events
              atomicMax(&tb.mm(sig)->x, ~d32);
              atomicMax(&tb.mm(sig)->y, d32);
            }
            if (old + d32 < old) atomicAdd(tb.sum_hi(sig), 1u);
            ok = true;
          }
        }
        if (!fits && live) {
          // the compact cell cannot take this event and the record is live: L2 atomics
          argus_cell* cl = reinterpret_cast<argus_cell*>(records + (size_t)cur_key * D.rec_bytes + D.cell_off) + sig;
          atomicAdd(reinterpret_cast<unsigned long long*>(&cl->count), 1ull);
          atomicAdd(reinterpret_cast<unsigned long long*>(&cl->sum_ns), d);
          atomicMin(reinterpret_cast<unsigned long long*>(&cl->min_ns), d);
          atomicMax(reinterpret_cast<unsigned long long*>(&cl->max_ns), d);
          atomicAdd(&cl->hist[argus_bucket64(d)], 1u);
          ok = true;
        }
      }
      // ---- spans of the folded events: warp-uniform fast path in registers, else ballot groups ------
      const uint32_t ph0 = __shfl_sync(FULL, phase, 0);
      if (__all_sync(FULL, ok && phase == ph0)) {
        if (ws.phase != ph0) { ws.flush(lane); ws.phase = ph0; }
        ws.mn = start < ws.mn ? start : ws.mn;
        ws.mx = end > ws.mx ? end : ws.mx;
        ws.n += 32u;                       // warp-uniform count
      } else {
        uint32_t todo = __ballot_sync(FULL, ok);
        while (todo) {
          const int leader = __ffs((int)todo) - 1;
          const uint32_t ph = __shfl_sync(FULL, phase, leader);
          const bool mine = ok && phase == ph;
          const uint32_t g2 = __ballot_sync(FULL, mine);
          const long long a = warp_min_i64(mine ? start : INT64_MAX);
          const long long b = warp_max_i64(mine ? end : INT64_MIN);
          if (lane == leader) {
            SpanAcc* sp = span_tab() + ph;
            atomicMin(&sp->mn, a);
            atomicMax(&sp->mx, b);
            atomicAdd(&sp->n, (unsigned long long)__popc(g2));
          }
          todo &= ~g2;
        }
      }
      if (ok) pending = false;
      if (!__any_sync(FULL, pending)) break;
      ws.flush(lane);
      const unsigned long long r = park<NC>(gl, pending, key, idx, cur_key, live);
      cur_key = (uint32_t)r; live = (uint32_t)(r >> 32) & 1u;
    }
  }
  // ---- out of events: keep joining the rendezvous until every warp is done ---------------------------
  ws.flush(lane);
  if (lane == 0) atomicAdd(&H->n_finished, 1u);
  for (;;) {
    const unsigned long long r = park<NC>(gl, false, KEY_NONE, KEY_NONE, cur_key, live);
    if (r & PARK_DONE) break;
    cur_key = (uint32_t)r; live = (uint32_t)(r >> 32) & 1u;
  }

  n_invalid = __reduce_add_sync(FULL, n_invalid);
  if (lane == 0 && n_invalid) atomicAdd(&counters[1], (unsigned long long)n_invalid);
  if (tid == 0) atomicAdd(&counters[0], (unsigned long long)n_ev);   // seen; valid = seen - invalid
}

template <int CW, int WPSTG>
cudaError_t launch_variant(argus_ctx* ctx, const argus_event* ev, uint64_t n, void* d_records,
                           cudaStream_t s) {
  constexpr int SPI = CW / WPSTG;
  constexpr size_t STAGE_BYTES = (size_t)WPSTG * 32 * 32;
  const size_t fixed = stage_off(ctx->dims.S);
  int K = (int)(((size_t)ctx->max_smem_optin - fixed) / STAGE_BYTES);
  if (K > MAXK) K = MAXK;
  if (K < 2 * SPI + 1) return cudaErrorInvalidConfiguration;
  const size_t smem_bytes = fixed + (size_t)K * STAGE_BYTES;
  cudaError_t e = cudaFuncSetAttribute(aggregate_seg_kernel<CW, WPSTG>,
                                       cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem_bytes);
  if (e != cudaSuccess) return e;
  int grid = ctx->tune_grid > 0 ? ctx->tune_grid : ctx->sm_count;
  // a CTA's slot counters hold 26 bits between flushes: bound the span of one CTA
  const uint64_t tile = (uint64_t)CW * 32;
  const uint64_t cap = (1ull << 26) - tile;
  uint64_t per_cta = (n + grid - 1) / grid;
  if (per_cta > cap) per_cta = cap;
  per_cta = (per_cta + tile - 1) / tile * tile;
  const uint64_t ctas = (n + per_cta - 1) / per_cta;
  aggregate_seg_kernel<CW, WPSTG><<<(unsigned)ctas, (CW + 1) * 32, smem_bytes, s>>>(
      reinterpret_cast<const uint4*>(ev), n, per_cta, static_cast<uint8_t*>(d_records), ctx->d_state,
      ctx->d_counters, ctx->dims, K);
  return cudaGetLastError();
}

}  // namespace

bool argus_seg_supported(const argus_ctx* ctx) {
  // default variant: 6 KB stages, 5 per iteration, at least 11 in the ring
  return (size_t)stage_off(ctx->dims.S) + (size_t)11 * 6144 <= (size_t)ctx->max_smem_optin;
}

cudaError_t argus_launch_aggregate_seg(argus_ctx* ctx, const argus_event* ev, uint64_t n,
                                       void* d_records, cudaStream_t s) {
  if (n == 0) return cudaSuccess;
  switch (ctx->tune_variant) {
    case 1: return launch_variant<30, 10>(ctx, ev, n, d_records, s);
    case 2: return launch_variant<30, 15>(ctx, ev, n, d_records, s);
    case 3: return launch_variant<28, 7>(ctx, ev, n, d_records, s);
    case 4: return launch_variant<30, 6>(ctx, ev, n, d_records, s);
    case 5: return launch_variant<31, 31>(ctx, ev, n, d_records, s);
    case 6: return launch_variant<24, 8>(ctx, ev, n, d_records, s);
    default: return launch_variant<30, 6>(ctx, ev, n, d_records, s);
  }
}
