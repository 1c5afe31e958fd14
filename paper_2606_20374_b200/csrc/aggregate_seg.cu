// aggregate_seg.cu — segmented aggregation kernel (NS (3): "hand-written sm_100a aggregation
// kernels ... coalesced 128-bit vectorised loads, with TMA ... staging into shared memory ...
// shared-memory-privatised per-block histograms and min/max/sum ... warp-shuffle segmented
// reductions where a block spans rank-step boundaries, and flush to global in one pass").
//
// Persistent CTAs (one, two or three per SM by table size) each walk a contiguous span of the event
// buffer.  Events arrive through a ring of shared-memory stages filled by 2-D tiled TMA loads
// (cp.async.bulk.tensor.2d over whole 128-byte rows of four events, 128-byte swizzle, mbarrier
// complete_tx, L2 evict-first) issued by a producer warp; each consumer lane takes one event per
// iteration into registers with two conflict-free LDS.128.
// The CTA keeps ONE (rank, step) table in shared memory at a time, 32 bytes per sig, laid out as
// structure-of-arrays so that random sigs spread over all 32 banks:
//   slots[S]  uint4: four histogram counters, DIRECT-MAPPED by bucket & 3
//   sum_lo[S], sum_hi[S] u32: the 64-bit sum with an explicit carry
//   mm[S]     u64 {~min : 32 | max : 32} (0 = empty cell)
// Invariant of a compact cell: bucket(max) - bucket(min) <= 3, so the (at most four) occupied
// buckets are consecutive and bucket & 3 names each of them uniquely — no tags, no lookup.  An
// event inside [min, max] (the common case, checked with one 64-bit load) can never break the
// invariant; an event that would extend the range goes through a 64-bit CAS that refuses the
// extension when the invariant would break.  Only native 32-bit shared atomics are used on the
// hot path (64-bit shared atomic adds are CAS loops on sm_100a).
// An event the compact cell cannot take (a range wider than four buckets: the second mode of a kernel
// whose durations "differ by several multiples" between positions) is RE-QUEUED: the lane
// appends {sig, duration} to its CTA's spill region (workspace) and goes on — span and counters are taken
// at once.  At the flush of the key, after the table has been written and cleared, the CTA folds the
// key's spilled events into the empty table, where the sig's remaining events open a window of their own,
// and merges that second table into the (now live) record with L2 reductions on the non-empty cells.  What
// the replay still refuses, events of 2^32 ns or more, and everything when the spill area is absent or
// full, is parked in the CTA's overflow list (global memory, workspace) and applied to the
// record with L2 reductions at the flush; when the record is already live it goes there at once.  When the
// (rank, step) key changes the table is flushed: the first CTA to reach a record claims it and
// writes the whole 160-byte cells with coalesced 128-bit stores (no read-modify-write, no separate
// identity fill); any later contribution to the same record merges with L2 reductions.  Correct
// for ANY event order; fast when events are grouped by (rank, step) (R18).
#include <cuda.h>
#include <stddef.h>

#include <type_traits>

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
  unsigned long long next;            // rendezvous request {lowest pending event index : 32 | its key : 32}
  uint32_t mode;                      // claim on the current key's record: LAZY = ours to write, LIVE, BUSY = another CTA's
  uint32_t n_finished;                // consumer warps that ran out of events
  uint32_t ovf_n;                     // events parked in this CTA's overflow list since the last flush
  uint32_t spill_n;                   // events this CTA re-queued into its spill region
  uint32_t n_refused;                 // events that took the overflow list or L2 atomics
  uint32_t n_requeued;                // events replayed from the spill region (a CTA's span holds < 2^26 events)
};
constexpr uint32_t OVF_CAP = ARGUS_OVF_CAP;   // entries of a CTA's overflow list (16 bytes each, workspace)
constexpr unsigned long long NEXT_NONE = ~0ull;
static_assert(sizeof(Hdr) <= HDR_BYTES, "header");

extern __shared__ __align__(1024) uint8_t smem[];   // 1024: the 128-byte swizzle atom of the TMA stages

// The compact table of one (rank, step), addressed by 32-bit offsets from the dynamic shared
// window: slots[S] uint4 | sum_lo[S] u32 | sum_hi[S] u32 | mm[S] uint2 {~min, max}.
struct Table {
  uint32_t S;
  __device__ __forceinline__ uint4* slots(uint32_t sig) const { return reinterpret_cast<uint4*>(smem + TAB_OFF) + sig; }
  __device__ __forceinline__ uint32_t* sum_lo(uint32_t sig) const { return reinterpret_cast<uint32_t*>(smem + TAB_OFF + 16u * S) + sig; }
  __device__ __forceinline__ uint32_t* sum_hi(uint32_t sig) const { return reinterpret_cast<uint32_t*>(smem + TAB_OFF + 20u * S) + sig; }
  __device__ __forceinline__ uint2* mm(uint32_t sig) const { return reinterpret_cast<uint2*>(smem + TAB_OFF + 24u * S) + sig; }
  // zero the cells of sigs [0, n): four arrays (S here is the compiled capacity, n <= S the live sigs)
  __device__ __forceinline__ void clear(uint32_t n, uint32_t t, uint32_t nt) const {
    const uint4 z = make_uint4(0u, 0u, 0u, 0u);
    uint4* a = slots(0);
    for (uint32_t i = t; i < n; i += nt) a[i] = z;
    uint4* b = reinterpret_cast<uint4*>(sum_lo(0));
    uint4* c = reinterpret_cast<uint4*>(sum_hi(0));
    for (uint32_t i = t; i < (n + 3u) / 4u; i += nt) { b[i] = z; c[i] = z; }
    uint4* d = reinterpret_cast<uint4*>(mm(0));
    for (uint32_t i = t; i < (n + 1u) / 2u; i += nt) d[i] = z;
  }
};
__device__ __forceinline__ Hdr* hdr() { return reinterpret_cast<Hdr*>(smem); }
__device__ __forceinline__ SpanAcc* span_tab() { return reinterpret_cast<SpanAcc*>(smem + HDR_BYTES); }

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
// 2-D tiled TMA load of one stage: rows of 128 bytes (4 events) starting at row `row`, written to
// shared memory with the 128-byte swizzle (16-byte chunk index XOR row & 7), which makes the
// consumers' per-lane LDS.128 of 32-byte records bank-conflict free.  Rows beyond the tensor are
// zero-filled and still count towards the transaction bytes.
__device__ __forceinline__ void tma_load_rows(uint32_t dst, const CUtensorMap* tmap, uint32_t row,
                                              uint32_t bar, uint64_t policy) {
  asm volatile(
      "cp.async.bulk.tensor.2d.shared::cluster.global.mbarrier::complete_tx::bytes.L2::cache_hint "
      "[%0], [%1, {%2, %3}], [%4], %5;" ::"r"(dst),
      "l"(tmap), "r"(0), "r"(row), "r"(bar), "l"(policy)
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
  uint4* ovf;             // this CTA's overflow list: {sig, 0, duration lo, duration hi} of events the compact cell refused
  uint2* spill;           // this CTA's spill region: {sig, duration} of the current key's re-queued events
  uint32_t spill_cap;     // its capacity in events (0: no spill area)
  argus_dims D;
};

// ---- shared-memory accessors on 32-bit shared-window addresses (no generic-address arithmetic) ----
__device__ __forceinline__ uint4 lds128(uint32_t a) {
  uint4 v;
  asm volatile("ld.shared.v4.u32 {%0, %1, %2, %3}, [%4];" : "=r"(v.x), "=r"(v.y), "=r"(v.z), "=r"(v.w) : "r"(a));
  return v;
}
__device__ __forceinline__ uint2 lds64(uint32_t a) {
  uint2 v;
  asm volatile("ld.shared.v2.u32 {%0, %1}, [%2];" : "=r"(v.x), "=r"(v.y) : "r"(a));
  return v;
}
__device__ __forceinline__ uint32_t lds32(uint32_t a) {
  uint32_t v;
  asm volatile("ld.shared.u32 %0, [%1];" : "=r"(v) : "r"(a));
  return v;
}
__device__ __forceinline__ void reds_add(uint32_t a, uint32_t v) {
  asm volatile("red.shared.add.u32 [%0], %1;" ::"r"(a), "r"(v) : "memory");
}
__device__ __forceinline__ void reds_max(uint32_t a, uint32_t v) {
  asm volatile("red.shared.max.u32 [%0], %1;" ::"r"(a), "r"(v) : "memory");
}
__device__ __forceinline__ void reds_max_if(uint32_t a, uint32_t v, bool p) {   // predicated: no branch
  asm volatile("{\n.reg .pred q;\nsetp.ne.u32 q, %2, 0;\n@q red.shared.max.u32 [%0], %1;\n}" ::"r"(a), "r"(v),
               "r"((uint32_t)p)
               : "memory");
}
__device__ __forceinline__ uint32_t atoms_add(uint32_t a, uint32_t v) {
  uint32_t o;
  asm volatile("atom.shared.add.u32 %0, [%1], %2;" : "=r"(o) : "r"(a), "r"(v) : "memory");
  return o;
}
__device__ __forceinline__ unsigned long long atoms_cas64(uint32_t a, unsigned long long cmp,
                                                          unsigned long long val) {
  unsigned long long o;
  asm volatile("atom.shared.cas.b64 %0, [%1], %2, %3;" : "=l"(o) : "r"(a), "l"(cmp), "l"(val) : "memory");
  return o;
}
__device__ __forceinline__ uint32_t bucket32(uint32_t d) {   // R4 for d < 2^32: floor(log2 d), 0 for d <= 1
  uint32_t b;
  asm("bfind.u32 %0, %1;" : "=r"(b) : "r"(d | 1u));     // bit position of the leading one (FLO)
  return b;
}

// Rare path of the compact cell: the event's duration d lies outside the cell's [min, max] (or the
// cell is empty).  Extend the range with a 64-bit CAS unless that would spread the cell over more
// than four consecutive buckets; returns false then (the event takes the global path instead).
__device__ __noinline__ bool mm_extend(uint32_t a_mm, uint32_t d) {
  const uint2 o2 = lds64(a_mm);
  unsigned long long old = ((unsigned long long)o2.y << 32) | o2.x;
  for (;;) {
    const uint32_t nmin = (uint32_t)old, mx = (uint32_t)(old >> 32);
    const uint32_t nn = nmin > ~d ? nmin : ~d, nx = mx > d ? mx : d;
    if (bucket32(nx) - bucket32(~nn) > 3u) return false;
    const unsigned long long nw = ((unsigned long long)nx << 32) | nn;
    if (nw == old) return true;
    const unsigned long long prev = atoms_cas64(a_mm, old, nw);
    if (prev == old) return true;
    old = prev;
  }
}

// One event straight into the LIVE global record (the compact cell refused it).
__device__ __noinline__ void global_cell_add(uint8_t* records, const argus_dims& D, uint32_t key,
                                             uint32_t sig, unsigned long long d) {
  argus_cell* cl = reinterpret_cast<argus_cell*>(records + (size_t)key * D.rec_bytes + D.cell_off) + sig;
  atomicAdd(reinterpret_cast<unsigned long long*>(&cl->count), 1ull);
  atomicAdd(reinterpret_cast<unsigned long long*>(&cl->sum_ns), d);
  if (D.sums) atomicAdd(&D.sums[(size_t)key * D.S + sig], d);
  atomicMin(reinterpret_cast<unsigned long long*>(&cl->min_ns), d);
  atomicMax(reinterpret_cast<unsigned long long*>(&cl->max_ns), d);
  atomicAdd(&cl->hist[argus_bucket64(d)], 1u);
}

__device__ __forceinline__ void bar_consumers(int n) {   // named barrier 1: consumer warps only
  asm volatile("bar.sync 1, %0;" ::"r"(n) : "memory");
}
__device__ __forceinline__ void mbar_arrive(uint32_t bar) {
  asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(bar) : "memory");
}

// The compact-cell update of one event (sig, d32 < 2^32) outside the hot loop (the replay of re-queued
// events): same protocol as ARGUS_COMPACT_ADD in the kernel.  True if the cell took the event.
template <uint32_t SCAP>
__device__ __forceinline__ bool compact_add(uint32_t sbase, uint32_t sig, uint32_t d32) {
  const uint32_t a_slots = sbase + TAB_OFF, a_m = a_slots + 24u * SCAP + sig * 8u;
  const uint2 m = lds64(a_m);
  const uint32_t nd = ~d32, b = bucket32(d32);
  bool took = (b >= bucket32(~m.x)) & (b <= bucket32(m.y));
  reds_max_if(a_m, nd, took & (nd > m.x));
  reds_max_if(a_m + 4u, d32, took & (d32 > m.y));
  if (!took) took = mm_extend(a_m, d32);
  if (took) {
    reds_add(a_slots + sig * 16u + ((b & 3u) << 2), 1u);
    const uint32_t old = atoms_add(a_slots + 16u * SCAP + sig * 4u, d32);
    if (old > nd) reds_add(a_slots + 20u * SCAP + sig * 4u, 1u);
  }
  return took;
}

// The non-empty cells of the shared table into the LIVE record `key` with L2 reductions.
template <int NC, uint32_t SCAP>
__device__ __forceinline__ void merge_cells(uint8_t* rec, const argus_dims& D, uint32_t key) {
  const Table tb{SCAP};
  argus_cell* cells = reinterpret_cast<argus_cell*>(rec + D.cell_off);
  for (uint32_t sig = threadIdx.x; sig < D.S; sig += NC) {
    const uint4 s = *tb.slots(sig);
    const uint2 m = *tb.mm(sig);
    if ((m.x | m.y) != 0u) {
      const uint32_t sl[4] = {s.x, s.y, s.z, s.w};
      const uint32_t bl = bucket32(~m.x);
      unsigned long long cnt = 0;
#pragma unroll
      for (uint32_t k = 0; k < 4u; ++k) {
        if (sl[k]) {
          atomicAdd(&cells[sig].hist[bl + ((k - bl) & 3u)], sl[k]);   // the bucket >= bl with bucket & 3 == k
          cnt += sl[k];
        }
      }
      atomicAdd(reinterpret_cast<unsigned long long*>(&cells[sig].count), cnt);
      const unsigned long long sm = ((unsigned long long)*tb.sum_hi(sig) << 32) | *tb.sum_lo(sig);
      atomicAdd(reinterpret_cast<unsigned long long*>(&cells[sig].sum_ns), sm);
      if (D.sums) atomicAdd(&D.sums[(size_t)key * D.S + sig], sm);
      atomicMin(reinterpret_cast<unsigned long long*>(&cells[sig].min_ns), (unsigned long long)(~m.x));
      atomicMax(reinterpret_cast<unsigned long long*>(&cells[sig].max_ns), (unsigned long long)m.y);
    }
  }
}

// Flush the shared table of record `key` to global memory and clear it.  All NC consumer threads
// call between the rendezvous barrier (the table is final: every warp has flushed its WarpSpan)
// and the closing barrier of park().  The claim on the record was taken when the key was adopted
// (H->mode), so no global round trip sits on this path; the publication of a record we wrote
// (fence + state LIVE) is left to thread 0 alone, after the barrier that orders everybody's stores
// before it (fence cumulativity), while the others already clear the table.
template <int NC, uint32_t SCAP>
__device__ __noinline__ void flush_table(const Glob& g, uint32_t key, bool fence_all) {
  const int tid = threadIdx.x;
  const argus_dims& D = g.D;
  const Table tb{SCAP};
  Hdr* H = hdr();
  SpanAcc* spans = span_tab();
  uint32_t mode = *reinterpret_cast<volatile uint32_t*>(&H->mode);
  uint32_t n_ovf = *reinterpret_cast<volatile uint32_t*>(&H->ovf_n);
  n_ovf = n_ovf < OVF_CAP ? n_ovf : OVF_CAP;
  uint32_t n_sp = *reinterpret_cast<volatile uint32_t*>(&H->spill_n);   // re-queued events of this key
  n_sp = n_sp < g.spill_cap ? n_sp : g.spill_cap;
  if (mode == ARGUS_ST_BUSY) {
    // another (resident, running) CTA owns this record and is writing it: wait for it, then merge
    if (tid == 0) {
      while (atomicAdd(&g.state[key], 0u) != ARGUS_ST_LIVE) __nanosleep(128);
      __threadfence();
    }
    bar_consumers(NC);
    mode = ARGUS_ST_LIVE;
  }
  uint8_t* rec = g.records + (size_t)key * D.rec_bytes;
  if (mode == ARGUS_ST_LAZY) {
    // we own the record: write spans + cells once with plain streaming stores
    uint4* dst = reinterpret_cast<uint4*>(rec + D.span_off);
    const uint32_t span_chunks = 2u * (D.P + 1u);
    for (uint32_t ch = tid; ch < span_chunks; ch += NC) {
      uint4 v;
      const uint32_t k = ch >> 1;
      if (k < D.P && spans[k].n != 0ull) {
        const SpanAcc a = spans[k];
        v = (ch & 1u) ? make_uint4(0u, 0u, (uint32_t)a.n, (uint32_t)(a.n >> 32))
                      : make_uint4((uint32_t)a.mn, (uint32_t)((unsigned long long)a.mn >> 32),
                                   (uint32_t)a.mx, (uint32_t)((unsigned long long)a.mx >> 32));
      } else {
        v = argus_identity_chunk(D, ch);
      }
      __stcs(dst + ch, v);
    }
    // cells, as two coalesced streams of 16-byte chunks (the compact cell is re-read from shared
    // memory by every lane that needs it; lanes of one cell read the same words: broadcast).
    // (1) histogram chunks: 8 lanes per cell, a warp store covers 4 cells x 128 contiguous bytes.
    //     Counter j of a cell holds the bucket b >= bl with b & 3 == j, bl = bucket(min): bucket
    //     4k + j is live iff (4k + j - bl) mod 2^32 < 4 (counters beyond bucket(max) are 0 anyway).
    uint4* cdst = reinterpret_cast<uint4*>(rec + D.cell_off);
    for (uint32_t i = tid; i < 8u * D.S; i += NC) {
      const uint32_t sig = i >> 3, k4 = (i & 7u) << 2;
      const uint4 c = *tb.slots(sig);
      const uint32_t bl = bucket32(~tb.mm(sig)->x);
      uint4 v;
      v.x = (k4 - bl) < 4u ? c.x : 0u;
      v.y = (k4 + 1u - bl) < 4u ? c.y : 0u;
      v.z = (k4 + 2u - bl) < 4u ? c.z : 0u;
      v.w = (k4 + 3u - bl) < 4u ? c.w : 0u;
      __stcs(cdst + 10u * sig + 2u + (i & 7u), v);
    }
    // (2) head chunks {count, sum} {min, max}: 2 lanes per cell
    for (uint32_t i = tid; i < 2u * D.S; i += NC) {
      const uint32_t sig = i >> 1;
      const uint4 c = *tb.slots(sig);
      const uint2 m = *tb.mm(sig);
      uint4 v;
      if ((i & 1u) == 0u) {
        const unsigned long long cnt = (unsigned long long)c.x + c.y + c.z + c.w;
        v = make_uint4((uint32_t)cnt, (uint32_t)(cnt >> 32), *tb.sum_lo(sig), *tb.sum_hi(sig));
      } else {
        v = (m.x | m.y) == 0u ? make_uint4(0xFFFFFFFFu, 0xFFFFFFFFu, 0u, 0u) : make_uint4(~m.x, 0u, m.y, 0u);
      }
      __stcs(cdst + 10u * sig + (i & 1u), v);
    }
    if (D.sums) {      // the record's row of the sum plane, sig-contiguous
      unsigned long long* row = D.sums + (size_t)key * D.S;
      for (uint32_t sig = tid; sig < D.S; sig += NC)
        row[sig] = ((unsigned long long)*tb.sum_hi(sig) << 32) | *tb.sum_lo(sig);
    }
    if (fence_all || n_ovf || n_sp) __threadfence();   // L2 atomics on this record follow at once
  } else {
    // merge into a live record with L2 reductions (non-empty fields only)
    merge_cells<NC, SCAP>(rec, D, key);
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
  if (tid == 0 && mode == ARGUS_ST_LAZY) {
    __threadfence();
    atomicExch(&g.state[key], ARGUS_ST_LIVE);
  }
  // the events the compact cells refused since the last flush: straight into the record (written or
  // merged above) with L2 reductions; they commute with everybody else's, so publication need not wait
  for (uint32_t i = tid; i < n_ovf; i += NC) {
    const uint4 e = __ldcg(g.ovf + i);
    global_cell_add(g.records, D, key, e.x, ((unsigned long long)e.w << 32) | e.z);
  }
  if (tid == 0) H->ovf_n = 0u;
  tb.clear(D.S, (uint32_t)tid, (uint32_t)NC);
  for (uint32_t k = tid; k < D.P; k += NC) {
    spans[k].mn = INT64_MAX; spans[k].mx = INT64_MIN; spans[k].n = 0ull; spans[k].pad = 0ull;
  }
  if (n_sp) {   // CTA-uniform
    // Replay of the key's re-queued events (cells only: spans and counters were taken when they were set
    // aside).  The record is live (published above, or by its owner), the table is empty: a sig whose
    // events fell outside the first window opens a second one here; what even that refuses takes L2
    // reductions one by one.  Then the second table is merged into the record and cleared.
    bar_consumers(NC);                      // table cleared; every lane's spill stores are visible to the CTA
    const uint32_t sbase = smem_u32(smem);
    uint32_t refused = 0;
    for (uint32_t i = tid; i < n_sp; i += NC) {
      const uint2 e = __ldcg(g.spill + i);
      if (!compact_add<SCAP>(sbase, e.x, e.y)) {
        global_cell_add(g.records, D, key, e.x, (unsigned long long)e.y);
        ++refused;
      }
    }
    if (refused) atomicAdd(&H->n_refused, refused);
    bar_consumers(NC);
    merge_cells<NC, SCAP>(rec, D, key);
    if (tid == 0) { H->spill_n = 0u; H->n_requeued += n_sp; }
    bar_consumers(NC);                      // everybody has read its cells: clear
    tb.clear(D.S, (uint32_t)tid, (uint32_t)NC);
  }
}

// Rendezvous of all consumer warps (the only CTA-wide synchronisation of the steady state, taken
// once per (rank, step) boundary on grouped input): three barriers.  A warp comes here when it
// holds an event it cannot fold: another key than the table's, or an event that needs the global
// path while the record is not live yet; it posts {event index, key} with a 64-bit min.  Warps
// that see a request below their position, or have run out of events, join.  Then the table is
// flushed and the key of the lowest pending event becomes current; thread 0 claims its record
// (state LAZY -> BUSY) after the closing barrier, so the claim's round trip is off everybody's path.
// Result packed as {cur_key : 32 | live : 1 | all_done : 1} (by value: keeps the caller's state in registers).
constexpr unsigned long long PARK_LIVE = 1ull << 32, PARK_DONE = 1ull << 33;
template <int NC, uint32_t SCAP>
__device__ __noinline__ unsigned long long park(const Glob& gl, bool pending, uint32_t key,
                                                uint32_t my_idx, uint32_t cur_key, uint32_t live) {
  Hdr* H = hdr();
  const int tid = threadIdx.x;
  if (pending) atomicMin(&H->next, ((unsigned long long)my_idx << 32) | key);
  bar_consumers(NC);
  const unsigned long long nx = *reinterpret_cast<volatile unsigned long long*>(&H->next);
  const uint32_t fin = *reinterpret_cast<volatile uint32_t*>(&H->n_finished);
  const uint32_t nk = (uint32_t)nx;
  const bool none = nx == NEXT_NONE;
  if (none && fin != (uint32_t)(NC / 32)) {   // nobody holds a pending event, but not every warp is done
    bar_consumers(NC);
    return (unsigned long long)cur_key | (live ? PARK_LIVE : 0ull);
  }
  const bool same = !none && nk == cur_key;   // an overflow event asked for a live record
  if (cur_key != KEY_NONE) flush_table<NC, SCAP>(gl, cur_key, same);
  else bar_consumers(NC);                      // everybody has read H->next
  if (none) return PARK_DONE | cur_key;
  if (tid == 0) H->next = NEXT_NONE;
  bar_consumers(NC);
  if (tid == 0) {
    // the claim on the (new) current record, consumed by the next flush (after its rendezvous barrier)
    H->mode = same ? ARGUS_ST_LIVE : atomicCAS(&gl.state[nk], ARGUS_ST_LAZY, ARGUS_ST_BUSY);
  }
  if (same) live = 1u;
  else { cur_key = nk; live = 0u; }
  return (unsigned long long)cur_key | (live ? PARK_LIVE : 0ull);
}

// CW consumer warps + 1 producer warp.  Stage = WPSTG warps' worth of events (WPSTG KB).
// Ring depth for a table capacity SCAP and a stage of stage_bytes: everything left of the 227 KB a CTA
// may use, capped at MAXK, rounded down to a multiple of the stages taken per iteration (a warp
// group then always returns to the slots it released itself, so the parity it waits for can never
// alias a fill two rounds behind: bulk copies of different stages may complete out of order).
constexpr uint32_t SMEM_MAX = 232448;          // 227 KB: the opt-in limit of one CTA on sm_100
constexpr uint32_t ARGUS_SEG_MAX_SIGS = 5120;   // largest table capacity that still leaves a 6-stage ring
// MINB CTAs share an SM (228 KB, 1 KB of it reserved per CTA): small tables leave room for several
// smaller CTAs, whose rendezvous and flushes then overlap with the streaming of their neighbours.
__host__ __device__ constexpr uint32_t smem_budget(int minb) { return 233472u / (uint32_t)minb - 1024u; }
__host__ __device__ constexpr int ring_depth(uint32_t scap, uint32_t stage_bytes, int spi, int minb) {
  int k = (int)((smem_budget(minb) - ((TAB_OFF + 32u * scap + 127u) & ~127u)) / stage_bytes);
  if (k > MAXK) k = MAXK;
  return k - k % spi;
}

// CW consumer warps + 1 producer warp; a stage = WPSTG warps' worth of events (WPSTG KB); the table
// layout is compiled for SCAP sigs (S <= SCAP), so every table address is base + sig * c + constant.
template <int CW, int WPSTG, uint32_t SCAP, int MINB>
__global__ void __launch_bounds__((CW + 1) * 32, MINB)
aggregate_seg_kernel(const __grid_constant__ CUtensorMap tmap, const uint4* __restrict__ ev, uint64_t n,
                     uint64_t per_cta, uint8_t* records, uint32_t* state, unsigned long long* counters,
                     uint4* ovf, argus_dims D, uint2* spill, uint32_t spill_cap) {
  constexpr int K = ring_depth(SCAP, (uint32_t)WPSTG * 1024u, CW / WPSTG, MINB);
  static_assert(K >= 2 * (CW / WPSTG), "ring too shallow for this geometry");
  constexpr int NC = CW * 32;            // consumer threads
  constexpr int SUBE = WPSTG * 32;       // events per stage
  constexpr int SPI = CW / WPSTG;        // stages per iteration
  static_assert(CW % WPSTG == 0, "geometry");
  Glob gl;
  gl.records = records; gl.state = state; gl.D = D;
  gl.ovf = ovf + (size_t)blockIdx.x * OVF_CAP;
  gl.spill = spill + (size_t)blockIdx.x * spill_cap; gl.spill_cap = spill_cap;
  const Table tb{SCAP};
  Hdr* H = hdr();
  constexpr uint32_t stages = (TAB_OFF + 32u * SCAP + 127u) & ~127u;   // byte offset of the stage ring in smem

  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  const uint64_t e0 = (uint64_t)blockIdx.x * per_cta;
  if (e0 >= n) return;
  const uint64_t e1 = (e0 + per_cta < n) ? e0 + per_cta : n;
  const uint32_t n_ev = (uint32_t)(e1 - e0);
  const uint32_t n_sub = (n_ev + SUBE - 1) / SUBE;
  const uint32_t n_iter = (n_ev + NC - 1) / NC;

  if (tid == 0) {
    for (int k = 0; k < K; ++k) {
      mbar_init(smem_u32(&H->full[k]), 1u);
      mbar_init(smem_u32(&H->empty[k]), (uint32_t)WPSTG);
    }
    H->next = NEXT_NONE; H->mode = ARGUS_ST_LIVE; H->n_finished = 0u; H->ovf_n = 0u; H->spill_n = 0u; H->n_refused = 0u; H->n_requeued = 0u;
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
  }
  {
    tb.clear(D.S, (uint32_t)tid, (uint32_t)(CW + 1) * 32u);
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
      const uint64_t rows_total = n >> 2;                 // whole 128-byte rows of the buffer: the tensor
      const uint64_t row_cta = e0 >> 2;                   // e0 is a multiple of the tile, hence of 4
      for (uint32_t s = 0; s < n_sub; ++s) {
        if (round) mbar_wait(smem_u32(&H->empty[slot]), (round - 1u) & 1u);
        const uint32_t bar = smem_u32(&H->full[slot]);
        const uint64_t row = row_cta + (uint64_t)s * (SUBE / 4);
        if (row < rows_total) {
          mbar_expect_tx(bar, (uint32_t)SUBE * 32u);
          tma_load_rows(smem_u32(smem + stages + slot * (SUBE * 32u)), &tmap, (uint32_t)row, bar, policy);
        } else {
          mbar_arrive(bar);      // only the last < 4 events live here: the consumers load them directly
        }
        if (++slot == (uint32_t)K) { slot = 0; ++round; }
      }
    }
    return;
  }

  // ---- consumer warps -----------------------------------------------------------------------------
  // All shared-memory traffic of the hot loop goes through 32-bit shared-window addresses.
  uint32_t sbase = smem_u32(smem);
  asm volatile("mov.u32 %0, %0;" : "+r"(sbase));   // opaque: keep it in a register, do not rematerialise
  const uint32_t a_slots = sbase + TAB_OFF, a_sumlo = a_slots + 16u * SCAP, a_sumhi = a_slots + 20u * SCAP,
                 a_mm = a_slots + 24u * SCAP;
  const uint32_t a_ring = sbase + stages, ring_bytes = (uint32_t)K * (uint32_t)(SUBE * 32);
  const uint32_t a_nextidx = sbase + (uint32_t)offsetof(Hdr, next) + 4u;   // high word: the requested index
  const uint32_t bar_ring = (uint32_t)K * 8u;     // bytes of full[0..K)
  constexpr uint32_t EMPTY_OFF = MAXK * 8u;          // empty[k] sits MAXK*8 bytes after full[k]
  WarpSpan ws;
  ws.reset();
  uint32_t cur_key = KEY_NONE, live = 0u;
  uint32_t cur_rank = 0u, cur_step = 0u, s_eff = 0u;   // s_eff = 0 while no key is current: nothing is accepted
  uint32_t n_invalid = 0;
  const uint32_t grp = (uint32_t)warp / WPSTG, wis = (uint32_t)warp % WPSTG;   // stage group, warp in stage
  const uint32_t slot0 = grp % (uint32_t)K;
  uint32_t par = (grp / (uint32_t)K) & 1u;
  uint32_t a_bar = sbase + (uint32_t)offsetof(Hdr, full) + slot0 * 8u;      // full[slot] of this iteration
  const uint32_t a_bar_end = sbase + (uint32_t)offsetof(Hdr, full) + bar_ring;
  // this lane's record in a stage: row (lane >> 2) of the warp's 8 rows, 16-byte chunks 2q and 2q + 1
  // (q = lane & 3), each XOR-swizzled with the row number: lo at a_ev, hi at a_ev ^ 16
  uint32_t a_ev = a_ring + slot0 * (uint32_t)(SUBE * 32) + wis * 1024u + ((uint32_t)lane >> 2) * 128u +
                  ((((uint32_t)lane & 3u) * 2u) ^ ((uint32_t)lane >> 2)) * 16u;
  uint32_t s = grp;                              // this warp's stage (tail iteration only)
  uint32_t my_pos = (uint32_t)warp * 32u;        // first event of this warp's chunk

#define ARGUS_ADOPT(r)                                                              \
  do {                                                                              \
    cur_key = (uint32_t)(r); live = (uint32_t)((r) >> 32) & 1u;                     \
    if (cur_key != KEY_NONE) {                                                      \
      cur_rank = cur_key / D.T; cur_step = D.step_base + (cur_key - cur_rank * D.T); \
      s_eff = D.S;                                                                  \
    } else { s_eff = 0u; }                                                          \
  } while (0)

  // The compact-cell update of one event (sig, d32 < 2^32): true if the cell took it.
  //   bucket(d) inside the cell's bucket range [bucket(min), bucket(max)]: the invariant cannot break.
  //     Two PREDICATED 32-bit max reductions extend min / max when d lies outside [min, max]; no
  //     branch: with 10-20 % of the events extending their cell (the k-th event of a cell sets a
  //     record with probability 2/k) nearly every warp holds such a lane, and a divergent path here
  //     cost a sixth of the kernel's instructions.
  //   else (first event of a cell, or a new bucket): one 64-bit CAS from the loaded state to the
  //     extended one, unless the range would spread over more than four buckets; mm_extend retries
  //     under contention and refuses when the invariant would break.
#define ARGUS_COMPACT_ADD(took)                                                          \
  do {                                                                                   \
    const uint32_t a_m = a_mm + sig * 8u;                                                \
    const uint2 m = lds64(a_m);                                                          \
    const uint32_t nd = ~d32, b = bucket32(d32);                                         \
    took = (b >= bucket32(~m.x)) & (b <= bucket32(m.y));   /* false for an empty cell */ \
    reds_max_if(a_m, nd, took & (nd > m.x));                                             \
    reds_max_if(a_m + 4u, d32, took & (d32 > m.y));                                      \
    if (!took) {                                                                         \
      const uint32_t nn = m.x > nd ? m.x : nd, nx = m.y > d32 ? m.y : d32;               \
      if (bucket32(nx) - bucket32(~nn) <= 3u) {                                          \
        const unsigned long long was = ((unsigned long long)m.y << 32) | m.x;            \
        took = atoms_cas64(a_m, was, ((unsigned long long)nx << 32) | nn) == was;        \
        if (!took) took = mm_extend(a_m, d32);                                           \
      }                                                                                  \
    }                                                                                    \
    if (took) {                                                                          \
      reds_add(a_slots + sig * 16u + ((b & 3u) << 2), 1u);                               \
      const uint32_t old = atoms_add(a_sumlo + sig * 4u, d32);                           \
      if (old > nd) reds_add(a_sumhi + sig * 4u, 1u);   /* old + d32 carried */          \
    }                                                                                    \
  } while (0)

  // A refused event of the current key (d < 2^32) is appended as {sig, duration} to this CTA's spill region
  // and replayed at the flush of the key; its span and its place in the counters are taken here.
#define ARGUS_SPILL(okv)                                          \
  do {                                                           \
    if (spill_cap != 0u) {                                       \
      const uint32_t sp_ = atomicAdd(&H->spill_n, 1u);           \
      if (sp_ < spill_cap) {                                     \
        gl.spill[sp_] = make_uint2(sig, d32);                    \
        okv = true;                                              \
      }                                                          \
    }                                                            \
  } while (0)

  const uint32_t n_full = n_ev / (uint32_t)NC;   // iterations in which every lane of every warp has an event
  // One iteration of a consumer warp.  TAIL = the ragged last iteration (stage or lanes may be missing).
  auto body = [&](auto tail_c) {
    constexpr bool TAIL = decltype(tail_c)::value;
    // ---- load: one event per lane, stage -> registers; release the stage at once --------------------
    bool have = true, mine = true;
    if (TAIL) {
      have = s < n_sub;                          // this warp's stage exists (warp-uniform)
      mine = have && my_pos + (uint32_t)lane < n_ev;
    }
    // While a warp waits for data it watches the rendezvous request: a warp beyond the requested
    // position joins the rendezvous BEFORE taking its next chunk (a parked warp keeps its next
    // stage unreleased, which may stall the in-order producer, so nobody may wait for data while
    // others wait for him).  Warps before that position go on: their stages are always issued.
    if (have && !mbar_try_wait(a_bar, par)) {
      do {
        if (lds32(a_nextidx) < my_pos) {
          ws.flush(lane);
          const unsigned long long r = park<NC, SCAP>(gl, false, KEY_NONE, KEY_NONE, cur_key, live);
          ARGUS_ADOPT(r);
        }
      } while (!mbar_try_wait(a_bar, par));
    }
    uint4 lo, hi;
    if (have) {
      lo = lds128(a_ev);
      hi = lds128(a_ev ^ 16u);
      if (TAIL) {
        // the last n % 4 events of the buffer are not part of the tensor (whole 128-byte rows only)
        const uint64_t g = e0 + my_pos + (uint32_t)lane;
        if (g >= (n & ~3ull) && g < n) { lo = __ldg(ev + 2 * g); hi = __ldg(ev + 2 * g + 1); }
      }
    } else {
      lo = make_uint4(0u, 0u, 0u, 0u); hi = lo;
    }
    const uint32_t a_rel = a_bar + EMPTY_OFF;     // released below, once every lane's loads have landed
    a_bar += (uint32_t)(SPI * 8); a_ev += (uint32_t)(SPI * SUBE * 32);
    if (a_bar >= a_bar_end) { a_bar -= bar_ring; par ^= 1u; a_ev -= ring_bytes; }
    if (TAIL) s += SPI;
    my_pos += NC;

    // ---- decode.  Fast test first: the event belongs to the current key and fits a compact cell
    // (same rank and step words as the current key, sig and phase in range, both timestamps
    // non-negative, 0 <= end - start < 2^32).  Everything else is sorted out on the slow side.
    const uint32_t sig = lo.z, phase = lo.w >> 16;
    const long long start = (long long)(((unsigned long long)hi.y << 32) | hi.x);
    const long long end = (long long)(((unsigned long long)hi.w << 32) | hi.z);
    const unsigned long long d = (unsigned long long)(end - start);
    const uint32_t d32 = (uint32_t)d;
    bool fast = mine & (lo.x == cur_rank) & (lo.y == cur_step) & (sig < s_eff) & (phase < D.P) &
                ((int)(hi.y | hi.w) >= 0) & ((uint32_t)(d >> 32) == 0u);
    bool pending, ok = false, tried = false;
    uint32_t key = cur_key;
    const bool all_fast = __all_sync(FULL, fast);
    // Release the stage only now: the vote above consumed both halves of every lane's record, so
    // all 32 lanes' LDS have returned.  (An arrive issued right behind the loads can overtake
    // them in a congested shared-memory pipe; with a short ring the refill then lands under a
    // pending load — seen as records whose second half belonged to another event.)
    if (have && lane == 0) mbar_arrive(a_rel);
    if (all_fast) {
      // ---- hot path: the whole warp folds into the current table -------------------------------------
      ARGUS_COMPACT_ADD(ok);
      if (!ok) ARGUS_SPILL(ok);
      if (__all_sync(FULL, ok && phase == ws.phase)) {
        ws.mn = start < ws.mn ? start : ws.mn;
        ws.mx = end > ws.mx ? end : ws.mx;
        ws.n += 32u;                       // warp-uniform count
        return;
      }
      if (__all_sync(FULL, ok) && !__all_sync(FULL, phase == __shfl_sync(FULL, phase, 0))) {
        // every event folded, phases mixed inside the warp (input that was grouped by key but not by time:
        // the output of the grouping pass): the shared span accumulators lane by lane, nothing else to do
        SpanAcc* sp = span_tab() + phase;
        if (start < *reinterpret_cast<volatile long long*>(&sp->mn)) atomicMin(&sp->mn, start);
        if (end > *reinterpret_cast<volatile long long*>(&sp->mx)) atomicMax(&sp->mx, end);
        atomicAdd(reinterpret_cast<uint32_t*>(&sp->n), 1u);
        return;
      }
      pending = true; tried = true;        // a refused event or a phase change: general handling below
    } else {
      // full validity (R2, R3) of the lanes that failed the fast test
      pending = mine && argus_event_key(D, lo.x, lo.y, sig, phase, start, end, key);
      n_invalid += (mine && !pending) ? 1u : 0u;
      fast = pending && key == cur_key && (uint32_t)(d >> 32) == 0u;
    }

    const uint32_t idx = my_pos - (uint32_t)NC + (uint32_t)lane;   // position of this lane's event
    for (;;) {
      // ---- cells -----------------------------------------------------------------------------------
      if (!tried) {
        ok = false;
        if (fast) {
          ARGUS_COMPACT_ADD(ok);
          if (!ok) ARGUS_SPILL(ok);
        }
      }
      tried = false;
      if (!ok && pending && key == cur_key) {
        // the compact cell cannot take this event: L2 atomics if the record is live, else the CTA's
        // overflow list (applied at the flush); a full list asks for a live record at the rendezvous
        if (live) {
          global_cell_add(records, D, cur_key, sig, d);
          atomicAdd(&H->n_refused, 1u);
          ok = true;
        } else {
          const uint32_t oi = atomicAdd(&H->ovf_n, 1u);
          if (oi < OVF_CAP) {
            gl.ovf[oi] = make_uint4(sig, 0u, d32, (uint32_t)(d >> 32));
            atomicAdd(&H->n_refused, 1u);
            ok = true;
          }
        }
      }
      // ---- spans of the folded events.  A warp whose 32 events share one phase keeps the span in
      // registers; a warp with mixed phases (ungrouped or boundary input) updates the shared
      // accumulators lane by lane: test min/max with a plain load first (they rarely improve after
      // the first few events), count with a 32-bit add (a CTA's span holds < 2^26 events: no carry).
      {
        const uint32_t ph0 = __shfl_sync(FULL, phase, 0);
        if (__all_sync(FULL, ok && phase == ph0)) {
          if (ph0 != ws.phase) { ws.flush(lane); ws.phase = ph0; }
          ws.mn = start < ws.mn ? start : ws.mn;
          ws.mx = end > ws.mx ? end : ws.mx;
          ws.n += 32u;
        } else if (ok) {
          SpanAcc* sp = span_tab() + phase;
          if (start < *reinterpret_cast<volatile long long*>(&sp->mn)) atomicMin(&sp->mn, start);
          if (end > *reinterpret_cast<volatile long long*>(&sp->mx)) atomicMax(&sp->mx, end);
          atomicAdd(reinterpret_cast<uint32_t*>(&sp->n), 1u);
        }
      }
      if (ok) { pending = false; fast = false; }
      if (!__any_sync(FULL, pending)) break;
      ws.flush(lane);
      const unsigned long long r = park<NC, SCAP>(gl, pending, key, idx, cur_key, live);
      ARGUS_ADOPT(r);
      fast = pending && key == cur_key && (uint32_t)(d >> 32) == 0u;
    }
  };
#pragma unroll 1
  for (uint32_t it = 0; it < n_full; ++it) body(std::false_type{});
  if (n_iter > n_full) { s = grp + n_full * (uint32_t)SPI; body(std::true_type{}); }
#undef ARGUS_COMPACT_ADD
#undef ARGUS_SPILL
  // ---- out of events: keep joining the rendezvous until every warp is done ---------------------------
  ws.flush(lane);
  if (lane == 0) atomicAdd(&H->n_finished, 1u);
  for (;;) {
    const unsigned long long r = park<NC, SCAP>(gl, false, KEY_NONE, KEY_NONE, cur_key, live);
    if (r & PARK_DONE) break;
    cur_key = (uint32_t)r; live = (uint32_t)(r >> 32) & 1u;
  }
#undef ARGUS_ADOPT

  n_invalid = __reduce_add_sync(FULL, n_invalid);
  if (lane == 0 && n_invalid) atomicAdd(&counters[1], (unsigned long long)n_invalid);
  if (tid == 0) {
    // H->* are final: every warp has passed the last rendezvous
    atomicAdd(&counters[0], (unsigned long long)n_ev);   // seen; valid = seen - invalid
    const uint32_t nq = *reinterpret_cast<volatile uint32_t*>(&H->n_requeued);
    if (nq) atomicAdd(&counters[3], (unsigned long long)nq);
    const uint32_t nr = *reinterpret_cast<volatile uint32_t*>(&H->n_refused);
    if (nr) atomicAdd(&counters[2], (unsigned long long)nr);
  }
}

// shared-memory bytes of one geometry
template <int CW, int WPSTG, uint32_t SCAP, int MINB>
constexpr size_t geom_smem() {
  return ((TAB_OFF + 32u * SCAP + 127u) & ~127u) +
         (size_t)ring_depth(SCAP, (uint32_t)WPSTG * 1024u, CW / WPSTG, MINB) * ((size_t)WPSTG * 1024u);
}

template <int CW, int WPSTG, uint32_t SCAP, int MINB>
cudaError_t configure_cap() {
  static_assert(geom_smem<CW, WPSTG, SCAP, MINB>() <= smem_budget(MINB), "shared memory");
  return cudaFuncSetAttribute(aggregate_seg_kernel<CW, WPSTG, SCAP, MINB>,
                              cudaFuncAttributeMaxDynamicSharedMemorySize,
                              (int)geom_smem<CW, WPSTG, SCAP, MINB>());
}

// the events at `base` as a 2-D tensor of whole 128-byte rows (4 events), loaded a stage (box_rows rows) at a
// time with the 128-byte shared-memory swizzle
static cudaError_t encode_events(argus_ctx* ctx, const void* base, uint64_t rows, uint32_t box_rows, CUtensorMap* tmap) {
  typedef CUresult (*encode_fn)(CUtensorMap*, CUtensorMapDataType, cuuint32_t, void*, const cuuint64_t*,
                                const cuuint64_t*, const cuuint32_t*, const cuuint32_t*,
                                CUtensorMapInterleave, CUtensorMapSwizzle, CUtensorMapL2promotion,
                                CUtensorMapFloatOOBfill);
  const encode_fn encode = reinterpret_cast<encode_fn>(ctx->fn_tmap_encode);
  if (!encode) return cudaErrorNotSupported;
  const cuuint64_t dims[2] = {32u, rows ? rows : 1u};          // u32 elements per row, rows
  const cuuint64_t strides[1] = {128u};                        // bytes between rows
  const cuuint32_t box[2] = {32u, (cuuint32_t)box_rows};
  const cuuint32_t estr[2] = {1u, 1u};
  // rows == 0: the map is never used (the producer only arrives), but it must still encode; point
  // it at the buffer with a single row that is never fetched
  const CUresult r = encode(tmap, CU_TENSOR_MAP_DATA_TYPE_UINT32, 2u, const_cast<void*>(base), dims,
                            strides, box, estr, CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_128B,
                            CU_TENSOR_MAP_L2_PROMOTION_L2_256B, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
  return r == CUDA_SUCCESS ? cudaSuccess : cudaErrorInvalidValue;
}

template <int CW, int WPSTG, uint32_t SCAP, int MINB>
cudaError_t launch_cap(argus_ctx* ctx, const argus_event* ev, uint64_t n, void* d_records, cudaStream_t s) {
  constexpr size_t smem_bytes = geom_smem<CW, WPSTG, SCAP, MINB>();
  int grid = ctx->tune_grid > 0 ? ctx->tune_grid : ctx->sm_count * MINB;
  if (grid > (int)ARGUS_MAX_SEG_CTAS) grid = (int)ARGUS_MAX_SEG_CTAS;
  // the u32 histogram counters of a CTA must not wrap between flushes: bound the span of one CTA
  const uint64_t tile = (uint64_t)CW * 32;
  const uint64_t cap = (1ull << 26) - tile;
  uint64_t per_cta = (n + grid - 1) / grid;
  if (per_cta > cap) per_cta = cap;
  per_cta = (per_cta + tile - 1) / tile * tile;
  const uint64_t ctas = (n + per_cta - 1) / per_cta;     // <= max(grid, 2^32 / 2^26 + 1) <= ARGUS_MAX_SEG_CTAS
  // the last n % 4 events are not part of the tensor: the consumers read them directly
  CUtensorMap tmap;
  cudaError_t e = encode_events(ctx, ev, n >> 2, (uint32_t)(WPSTG * 8), &tmap);
  if (e != cudaSuccess) return e;
  // spill regions: one per CTA, 8 bytes per re-queued event of the CTA's CURRENT key (0: refused events go to
  // the overflow lists)
  uint64_t scap = ctx->d_spill ? (uint64_t)ctx->cfg.max_spill_events / ctas : 0u;
  if (scap > per_cta) scap = per_cta;
  aggregate_seg_kernel<CW, WPSTG, SCAP, MINB><<<(unsigned)ctas, (CW + 1) * 32, smem_bytes, s>>>(
      tmap, reinterpret_cast<const uint4*>(ev), n, per_cta, static_cast<uint8_t*>(d_records), ctx->d_state,
      ctx->d_counters, ctx->d_ovf, ctx->dims, reinterpret_cast<uint2*>(ctx->d_spill), (uint32_t)scap);
  ctx->n_kernels += 1;
  return cudaGetLastError();
}

}  // namespace

// Geometry by table size: as many CTAs per SM as the table leaves room for (three CTAs of 8 consumer warps
// for S <= 1024, two 15-warp CTAs for S <= 2048, else one 30-warp CTA), compiled per table capacity.
// Warp w of a CTA runs on scheduler w mod 4, and the kernel is close to issue-bound: with 8 consumer warps
// per CTA every scheduler of the SM gets 3 x 2 of them; 9 (the producer being the tenth) put 9 / 6 / 6 / 6
// on the four schedulers and the first one set the pace (mid 0.413 -> 0.382 ms, scale 1.853 -> 1.790 ms).
// An 8-warp stage (8 KB) keeps the single producer lane at one bulk copy per CTA iteration.
bool argus_seg_supported(const argus_ctx* ctx) {
  return ctx->dims.S <= ARGUS_SEG_MAX_SIGS && (size_t)ctx->max_smem_optin >= SMEM_MAX && ctx->fn_tmap_encode != nullptr;
}

cudaError_t argus_configure_seg(argus_ctx* ctx) {
  if (!argus_seg_supported(ctx)) return cudaSuccess;
  const uint32_t S = ctx->dims.S;
  if (S <= 512u) return configure_cap<8, 8, 512u, 3>();
  if (S <= 1024u) return configure_cap<8, 8, 1024u, 3>();
  if (S <= 2048u) return configure_cap<15, 5, 2048u, 2>();
  if (S <= 4096u) return configure_cap<30, 10, 4096u, 1>();
  return configure_cap<30, 10, ARGUS_SEG_MAX_SIGS, 1>();
}

cudaError_t argus_launch_aggregate_seg(argus_ctx* ctx, const argus_event* ev, uint64_t n,
                                       void* d_records, cudaStream_t s) {
  if (n == 0) return cudaSuccess;
  const uint32_t S = ctx->dims.S;
  if (S <= 512u) return launch_cap<8, 8, 512u, 3>(ctx, ev, n, d_records, s);
  if (S <= 1024u) return launch_cap<8, 8, 1024u, 3>(ctx, ev, n, d_records, s);
  if (S <= 2048u) return launch_cap<15, 5, 2048u, 2>(ctx, ev, n, d_records, s);
  if (S <= 4096u) return launch_cap<30, 10, 4096u, 1>(ctx, ev, n, d_records, s);
  if (S <= ARGUS_SEG_MAX_SIGS) return launch_cap<30, 10, ARGUS_SEG_MAX_SIGS, 1>(ctx, ev, n, d_records, s);
  return cudaErrorInvalidConfiguration;
}
