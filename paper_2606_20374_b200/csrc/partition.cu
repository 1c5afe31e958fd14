// partition.cu — grouping pass for ungrouped input (BASELINE.json configs[3]: "records shuffled
// uniformly across rank-steps, so aggregation cannot rely on contiguous segments").
//
// Folding shuffled events straight into a dense table that is far larger than L2 costs several
// random 32-byte read-modify-writes in HBM per event (aggregate_global.cu: 6 G events/s).  Moving
// each record to its (rank, step) group first lets the segmented kernel run on contiguous segments.
// key = rank*T + step - step_base.  Three layouts of the pass, chosen per table geometry when the
// context is created; all buffers are areas of the caller's workspace:
//   two-level (R*T <= 24576, the default; second half of this file): count, scan, a coarse pass into
//             <= 256 bins of 16-byte packed events, a fine pass back to raw events per key, pad —
//             every tile counting-sorted in shared memory and written out as contiguous runs
//   single scatter, shared-memory cursors (R*T + 1 counters fit shared memory):
//     count   : every CTA owns a contiguous chunk of the buffer and counts its keys in a shared-memory
//               histogram (no global atomics), then writes its row H[cta][key]
//     offsets : per key, exclusive running sum over the CTAs (H[cta][key] becomes the CTA's offset
//               inside the key's group) and the group size total[key]
//     scan    : exclusive prefix sum of total in place (one CTA, running carry)
//     scatter : the same CTA re-reads its chunk with cursor[key] = total[key] + H[cta][key] in shared
//               memory: pos = atomicAdd(&cursor[key], 1); grouped[pos] = event (one 256-bit store)
//   single scatter, global cursors (anything larger): count and scatter use L2 atomics on one global
//             counter array (same results, slower)
// In the single-scatter layouts key-invalid events go to bin R*T, in the two-level layout invalid events
// are dropped and re-appear as padding: either way the segmented kernel still sees (and counts) every
// event of the call; sig / phase / timestamp validity is its business.
#include "argus_internal.cuh"

namespace {

__device__ __forceinline__ uint32_t group_key(const argus_dims& D, uint32_t rank, uint32_t step) {
  const uint32_t t = step - D.step_base;
  return (rank < D.R && t < D.T) ? rank * D.T + t : D.R * D.T;
}

// One event = one 32-byte sector: a single 256-bit store (sm_100) instead of two partial-sector writes.
__device__ __forceinline__ void store_event(uint4* dst, const uint4& lo, const uint4& hi) {
  asm volatile("st.global.v8.b32 [%0], {%1, %2, %3, %4, %5, %6, %7, %8};" ::"l"(dst), "r"(lo.x), "r"(lo.y),
               "r"(lo.z), "r"(lo.w), "r"(hi.x), "r"(hi.y), "r"(hi.z), "r"(hi.w)
               : "memory");
}

__global__ void __launch_bounds__(512)
partition_count_kernel(const uint4* __restrict__ ev, uint64_t n, argus_dims D, uint32_t* hist) {
  const uint64_t stride = (uint64_t)gridDim.x * blockDim.x;
  for (uint64_t i = (uint64_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += stride) {
    const uint4 lo = __ldg(ev + 2 * i);
    atomicAdd(&hist[group_key(D, lo.x, lo.y)], 1u);
  }
}

// in-place exclusive scan of hist[0..m) by one CTA of 1024 threads
__global__ void __launch_bounds__(1024)
partition_scan_kernel(uint32_t* hist, uint32_t m) {
  __shared__ uint32_t warp_sum[32];
  __shared__ uint32_t carry_s;
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  if (tid == 0) carry_s = 0u;
  __syncthreads();
  for (uint32_t base = 0; base < m; base += 1024u) {
    const uint32_t i = base + (uint32_t)tid;
    const uint32_t v = i < m ? hist[i] : 0u;
    uint32_t inc = v;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
      const uint32_t t = __shfl_up_sync(0xFFFFFFFFu, inc, o);
      if (lane >= o) inc += t;
    }
    if (lane == 31) warp_sum[warp] = inc;
    __syncthreads();
    if (warp == 0) {
      uint32_t w = warp_sum[lane], winc = w;
#pragma unroll
      for (int o = 1; o < 32; o <<= 1) {
        const uint32_t t = __shfl_up_sync(0xFFFFFFFFu, winc, o);
        if (lane >= o) winc += t;
      }
      warp_sum[lane] = winc - w;          // exclusive offset of each warp
    }
    __syncthreads();
    const uint32_t carry = carry_s;
    if (i < m) hist[i] = carry + warp_sum[warp] + inc - v;
    __syncthreads();
    if (tid == 1023) carry_s = carry + warp_sum[31] + inc;
    __syncthreads();
  }
}

__global__ void __launch_bounds__(512)
partition_scatter_kernel(const uint4* __restrict__ ev, uint64_t n, argus_dims D, uint32_t* cursor,
                         uint4* __restrict__ grouped) {
  const uint64_t stride = (uint64_t)gridDim.x * blockDim.x;
  for (uint64_t i = (uint64_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += stride) {
    const uint4 lo = ev[2 * i], hi = ev[2 * i + 1];
    const uint32_t pos = atomicAdd(&cursor[group_key(D, lo.x, lo.y)], 1u);
    store_event(grouped + 2 * (size_t)pos, lo, hi);
  }
}

// ---- shared-memory variant: per-CTA histograms, no global atomics -----------------------------------
extern __shared__ uint32_t s_bins[];

__global__ void __launch_bounds__(1024)
partition_count_smem_kernel(const uint4* __restrict__ ev, uint64_t n, uint64_t chunk, argus_dims D,
                            uint32_t m, uint32_t* __restrict__ H) {
  for (uint32_t k = threadIdx.x; k < m; k += blockDim.x) s_bins[k] = 0u;
  __syncthreads();
  const uint64_t e0 = (uint64_t)blockIdx.x * chunk;
  const uint64_t e1 = e0 + chunk < n ? e0 + chunk : n;
  for (uint64_t i = e0 + threadIdx.x; i < e1; i += blockDim.x) {
    const uint4 lo = __ldcs(ev + 2 * i);
    atomicAdd(&s_bins[group_key(D, lo.x, lo.y)], 1u);
  }
  __syncthreads();
  uint32_t* row = H + (size_t)blockIdx.x * m;
  for (uint32_t k = threadIdx.x; k < m; k += blockDim.x) row[k] = s_bins[k];
}

// H[c][k] := sum over c' < c of H[c'][k];  total[k] := sum over all c
__global__ void __launch_bounds__(256)
partition_offsets_kernel(uint32_t* __restrict__ H, uint32_t n_cta, uint32_t m, uint32_t* __restrict__ total) {
  const uint32_t k = blockIdx.x * blockDim.x + threadIdx.x;
  if (k >= m) return;
  uint32_t run = 0;
  for (uint32_t c = 0; c < n_cta; ++c) {
    const uint32_t v = H[(size_t)c * m + k];
    H[(size_t)c * m + k] = run;
    run += v;
  }
  total[k] = run;
}

__global__ void __launch_bounds__(1024)
partition_scatter_smem_kernel(const uint4* __restrict__ ev, uint64_t n, uint64_t chunk, argus_dims D,
                              uint32_t m, const uint32_t* __restrict__ H,
                              const uint32_t* __restrict__ start, uint4* __restrict__ grouped) {
  const uint32_t* row = H + (size_t)blockIdx.x * m;
  for (uint32_t k = threadIdx.x; k < m; k += blockDim.x) s_bins[k] = start[k] + row[k];
  __syncthreads();
  const uint64_t e0 = (uint64_t)blockIdx.x * chunk;
  const uint64_t e1 = e0 + chunk < n ? e0 + chunk : n;
  for (uint64_t i = e0 + threadIdx.x; i < e1; i += blockDim.x) {
    const uint4 lo = __ldcs(ev + 2 * i), hi = __ldcs(ev + 2 * i + 1);
    const uint32_t pos = atomicAdd(&s_bins[group_key(D, lo.x, lo.y)], 1u);
    store_event(grouped + 2 * (size_t)pos, lo, hi);
  }
}


// ==== two-level grouping (the default when R*T <= P2_MAX_KEYS) =========================================
// A single scatter into R*T groups leaves every CTA with thousands of open 32-byte write streams: L2
// evicts the lines before they fill and HBM sees row-missing sector writes (2.1 TB/s).
// Two levels of at most 256 bins each, every tile of 1024 events counting-sorted in shared memory and copied
// out as runs of whole lines reserved with ONE global atomic per (tile, bin), stream instead:
//   count   valid events per key (shared-memory histogram per CTA, merged with L2 atomics) and packable
//           events per coarse bin (key >> shift)
//   scan    key offsets (cursors of the final layout), coarse-bin offsets, tiles per coarse bin
//   coarse  raw events -> 16-byte packed events {sig : 13 | phase : 6 | key in bin : 13, duration u32,
//           start i64}, grouped by coarse bin.  Invalid events (R2, R3) are dropped here; a valid event whose
//           duration does not fit 32 bits goes straight to its final place with a per-key L2 atomic
//   fine    one coarse bin at a time: packed events -> raw 32-byte events (stream id 0: not part of the
//           method, R16) grouped by key
//   pad     the n - n_valid slots behind the grouped events become invalid records (rank 2^32 - 1), so that
//           the segmented kernel still sees and counts every event of the call
constexpr uint32_t P2_MAX_BINS = 256;

struct P2Small {          // small device-side state of one grouping pass (in the `part` area of the workspace)
  uint32_t n_valid;       // events that are grouped (everything else is padding)
  uint32_t n_tiles;       // tiles of the fine pass
  uint32_t pad[2];
  uint32_t chist[P2_MAX_BINS];          // packable events per coarse bin
  uint32_t cstart[P2_MAX_BINS + 1];     // first slot of each coarse bin in the coarse area
  uint32_t ccur[P2_MAX_BINS];           // cursors of the coarse pass
  uint32_t tiles_before[P2_MAX_BINS + 1];
};

__device__ __forceinline__ uint4 ldcs128(const uint4* p) { return __ldcs(p); }

// validity (R2, R3) + key of a raw event; also whether its duration fits 32 bits
__device__ __forceinline__ bool p2_decode(const argus_dims& D, const uint4& lo, const uint4& hi, uint32_t& key,
                                          bool& packable) {
  const long long start = (long long)(((unsigned long long)hi.y << 32) | hi.x);
  const long long end = (long long)(((unsigned long long)hi.w << 32) | hi.z);
  const bool ok = argus_event_key(D, lo.x, lo.y, lo.z, lo.w >> 16, start, end, key);
  packable = ((unsigned long long)(end - start) >> 32) == 0ull;
  return ok;
}

__global__ void __launch_bounds__(1024)
p2_count_kernel(const uint4* __restrict__ ev, uint64_t n, uint64_t chunk, argus_dims D, uint32_t shift,
                uint32_t* __restrict__ khist, P2Small* __restrict__ sm) {
  const uint32_t RT = D.R * D.T;
  uint32_t* s_c = s_bins + RT;                       // coarse counters behind the key counters
  for (uint32_t k = threadIdx.x; k < RT + P2_MAX_BINS; k += blockDim.x) s_bins[k] = 0u;
  __syncthreads();
  const uint64_t e0 = (uint64_t)blockIdx.x * chunk;
  const uint64_t e1 = e0 + chunk < n ? e0 + chunk : n;
  for (uint64_t i = e0 + threadIdx.x; i < e1; i += blockDim.x) {
    const uint4 lo = ldcs128(ev + 2 * i), hi = ldcs128(ev + 2 * i + 1);
    uint32_t key; bool packable;
    if (p2_decode(D, lo, hi, key, packable)) {
      atomicAdd(&s_bins[key], 1u);
      if (packable) atomicAdd(&s_c[key >> shift], 1u);
    }
  }
  __syncthreads();
  for (uint32_t k = threadIdx.x; k < RT; k += blockDim.x)
    if (s_bins[k]) atomicAdd(&khist[k], s_bins[k]);
  for (uint32_t k = threadIdx.x; k < P2_MAX_BINS; k += blockDim.x)
    if (s_c[k]) atomicAdd(&sm->chist[k], s_c[k]);
}

// exclusive block scan over 1024 threads (one value each); returns the prefix, the total in `total`
__device__ __forceinline__ uint32_t scan1024(uint32_t v, uint32_t* s_w, uint32_t& total) {
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  uint32_t inc = v;
#pragma unroll
  for (int o = 1; o < 32; o <<= 1) {
    const uint32_t t = __shfl_up_sync(0xFFFFFFFFu, inc, o);
    if (lane >= o) inc += t;
  }
  if (lane == 31) s_w[warp] = inc;
  __syncthreads();
  uint32_t before = 0u, all = 0u;
  for (int w = 0; w < (int)(blockDim.x >> 5); ++w) {
    const uint32_t x = s_w[w];
    if (w < warp) before += x;
    all += x;
  }
  __syncthreads();
  total = all;
  return before + inc - v;
}

// key offsets in place (khist[k] := first slot of key k in the grouped layout), coarse offsets, tile counts
__global__ void __launch_bounds__(1024)
p2_scan_kernel(uint32_t* khist, uint32_t RT, P2Small* sm, uint32_t fine_tile) {
  __shared__ uint32_t s_w[32];
  uint32_t carry = 0u;
  for (uint32_t base = 0; base < RT; base += 1024u) {
    const uint32_t i = base + threadIdx.x;
    const uint32_t v = i < RT ? khist[i] : 0u;
    uint32_t total;
    const uint32_t pre = scan1024(v, s_w, total);
    if (i < RT) khist[i] = carry + pre;
    carry += total;
  }
  if (threadIdx.x == 0) sm->n_valid = carry;
  {
    const uint32_t b = threadIdx.x;
    const uint32_t c = b < P2_MAX_BINS ? sm->chist[b] : 0u;
    uint32_t total, ttotal;
    const uint32_t pre = scan1024(c, s_w, total);
    const uint32_t tpre = scan1024((c + fine_tile - 1u) / fine_tile, s_w, ttotal);
    if (b < P2_MAX_BINS) { sm->cstart[b] = pre; sm->ccur[b] = pre; sm->tiles_before[b] = tpre; }
    if (b == 0) { sm->cstart[P2_MAX_BINS] = total; sm->tiles_before[P2_MAX_BINS] = ttotal; sm->n_tiles = ttotal; }
  }
}

template <uint32_t TILE>
struct P2SharedT {
  uint32_t cnt[P2_MAX_BINS];
  uint32_t off[P2_MAX_BINS];
  uint32_t gbase[P2_MAX_BINS];
  uint32_t rank[P2_MAX_BINS], step[P2_MAX_BINS];   // fine pass: (rank, step) of every key of the bin
  uint32_t w[32];
  uint32_t n_packed, unused;
  uint8_t binof[TILE];
};

// exclusive scan of cnt[0..256) by the first 256 threads (all threads of the CTA call; NT >= 256); also resets cnt
template <class SH>
__device__ __forceinline__ void p2_bins_scan(SH* S, uint32_t& my_cnt, uint32_t& my_pre) {
  const uint32_t t = threadIdx.x;
  const int lane = t & 31, warp = t >> 5;
  uint32_t c = t < P2_MAX_BINS ? S->cnt[t] : 0u;
  uint32_t inc = c;
#pragma unroll
  for (int o = 1; o < 32; o <<= 1) {
    const uint32_t x = __shfl_up_sync(0xFFFFFFFFu, inc, o);
    if (lane >= o) inc += x;
  }
  if (lane == 31 && warp < 8) S->w[warp] = inc;
  __syncthreads();
  uint32_t before = 0u;
  for (int w = 0; w < 8; ++w) if (w < warp) before += S->w[w];
  my_cnt = c; my_pre = before + inc - c;
  if (t < P2_MAX_BINS) { S->off[t] = my_pre; S->cnt[t] = 0u; }
}

template <uint32_t NT, uint32_t EPT, int MINB>
__global__ void __launch_bounds__(NT, MINB)
p2_coarse_kernel(const uint4* __restrict__ ev, uint64_t n, argus_dims D, uint32_t shift, uint32_t* __restrict__ kcur,
                 P2Small* __restrict__ sm, uint4* __restrict__ coarse, uint4* __restrict__ grouped) {
  constexpr uint32_t TILE = NT * EPT;
  typedef P2SharedT<TILE> SH;
  extern __shared__ __align__(16) uint8_t p2_smem[];
  SH* S = reinterpret_cast<SH*>(p2_smem);
  uint4* sorted = reinterpret_cast<uint4*>(p2_smem + ((sizeof(SH) + 15u) & ~15u));
  for (uint32_t k = threadIdx.x; k < P2_MAX_BINS; k += NT) S->cnt[k] = 0u;
  __syncthreads();
  const uint64_t n_tiles = (n + TILE - 1) / TILE;
  // software pipeline: the raw events of the NEXT tile are requested before this tile is sorted and copied out
  uint4 nlo[EPT], nhi[EPT];
#pragma unroll
  for (uint32_t j = 0; j < EPT; ++j) {
    const uint64_t i = (uint64_t)blockIdx.x * TILE + j * NT + threadIdx.x;
    nlo[j] = make_uint4(0u, 0u, 0u, 0u); nhi[j] = nlo[j];
    if (i < n) { nlo[j] = ldcs128(ev + 2 * i); nhi[j] = ldcs128(ev + 2 * i + 1); }
  }
  for (uint64_t tile = blockIdx.x; tile < n_tiles; tile += gridDim.x) {
    uint4 pk[EPT];
    uint32_t where[EPT];                          // bin << 16 | position inside the tile's bin; ~0 = not packed
    const uint64_t base = tile * TILE;
#pragma unroll
    for (uint32_t j = 0; j < EPT; ++j) {
      const uint64_t i = base + j * NT + threadIdx.x;
      where[j] = 0xFFFFFFFFu;
      if (i < n) {
        const uint4 lo = nlo[j], hi = nhi[j];
        uint32_t key; bool packable;
        if (p2_decode(D, lo, hi, key, packable)) {
          if (packable) {
            const uint32_t bin = key >> shift;
            pk[j] = make_uint4(lo.z | ((lo.w >> 16) << 13) | ((key - (bin << shift)) << 19), hi.z - hi.x, hi.x, hi.y);
            where[j] = (bin << 16) | atomicAdd(&S->cnt[bin], 1u);
          } else {
            // duration >= 2^32 ns: rare; straight to its final slot
            const uint32_t pos = atomicAdd(&kcur[key], 1u);
            store_event(grouped + 2 * (size_t)pos, make_uint4(lo.x, lo.y, lo.z, lo.w & 0xFFFF0000u), hi);
          }
        }
      }
    }
#pragma unroll
    for (uint32_t j = 0; j < EPT; ++j) {
      const uint64_t i = (tile + gridDim.x) * TILE + j * NT + threadIdx.x;
      if (i < n) { nlo[j] = ldcs128(ev + 2 * i); nhi[j] = ldcs128(ev + 2 * i + 1); }
    }
    __syncthreads();
    uint32_t c, pre;
    p2_bins_scan(S, c, pre);
    if (threadIdx.x < P2_MAX_BINS) S->gbase[threadIdx.x] = (c ? atomicAdd(&sm->ccur[threadIdx.x], c) : 0u) - pre;
    if (threadIdx.x == P2_MAX_BINS - 1u) S->n_packed = pre + c;   // packed events of this tile
    __syncthreads();
#pragma unroll
    for (uint32_t j = 0; j < EPT; ++j) {
      if (where[j] != 0xFFFFFFFFu) {
        const uint32_t bin = where[j] >> 16, slot = S->off[bin] + (where[j] & 0xFFFFu);
        sorted[slot] = pk[j];
        S->binof[slot] = (uint8_t)bin;
      }
    }
    __syncthreads();
    const uint32_t m = S->n_packed;
    for (uint32_t i = threadIdx.x; i < m; i += NT) coarse[(size_t)S->gbase[S->binof[i]] + i] = sorted[i];
    __syncthreads();
  }
}

template <uint32_t NT, uint32_t EPT, int MINB>
__global__ void __launch_bounds__(NT, MINB)
p2_fine_kernel(const uint4* __restrict__ coarse, argus_dims D, uint32_t shift, uint32_t* __restrict__ kcur,
               const P2Small* __restrict__ sm, uint4* __restrict__ grouped) {
  constexpr uint32_t TILE = NT * EPT;
  typedef P2SharedT<TILE> SH;
  extern __shared__ __align__(16) uint8_t p2_smem[];
  SH* S = reinterpret_cast<SH*>(p2_smem);
  uint4* sorted = reinterpret_cast<uint4*>(p2_smem + ((sizeof(SH) + 15u) & ~15u));   // [TILE][2]
  __shared__ uint32_t s_tb[P2_MAX_BINS + 1];
  for (uint32_t k = threadIdx.x; k <= P2_MAX_BINS; k += NT) s_tb[k] = sm->tiles_before[k];
  for (uint32_t k = threadIdx.x; k < P2_MAX_BINS; k += NT) S->cnt[k] = 0u;
  __syncthreads();
  const uint32_t n_tiles = s_tb[P2_MAX_BINS], RT = D.R * D.T, kpb = 1u << shift;
  uint32_t cur_bin = 0xFFFFFFFFu;
  // where tile `t` lives: its coarse bin (the last b with tiles_before[b] <= t), first slot and length
  auto locate = [&](uint32_t t, uint32_t& bin, uint32_t& s0, uint32_t& m) {
    uint32_t lo_b = 0u, hi_b = P2_MAX_BINS - 1u;
    while (lo_b < hi_b) {
      const uint32_t mid = (lo_b + hi_b + 1u) >> 1;
      if (s_tb[mid] <= t) lo_b = mid; else hi_b = mid - 1u;
    }
    bin = lo_b;
    s0 = sm->cstart[bin] + (t - s_tb[bin]) * TILE;
    const uint32_t s_end = sm->cstart[bin + 1u];
    m = s_end - s0 < TILE ? s_end - s0 : TILE;
  };
  // software pipeline: the packed events of the NEXT tile are requested before this tile is sorted and copied
  // out, so that their latency hides behind four barriers' worth of shared-memory work
  uint4 nx[EPT];
#pragma unroll
  for (uint32_t j = 0; j < EPT; ++j) nx[j] = make_uint4(0u, 0u, 0u, 0u);
  uint32_t nbin = 0u, ns0 = 0u, nm = 0u;
  if (blockIdx.x < n_tiles) {
    locate(blockIdx.x, nbin, ns0, nm);
#pragma unroll
    for (uint32_t j = 0; j < EPT; ++j) {
      const uint32_t i = j * NT + threadIdx.x;
      if (i < nm) nx[j] = ldcs128(coarse + (size_t)ns0 + i);
    }
  }
  for (uint32_t tile = blockIdx.x; tile < n_tiles; tile += gridDim.x) {
    const uint32_t bin = nbin, m = nm;
    if (bin != cur_bin) {                          // block-uniform
      cur_bin = bin;
      for (uint32_t j = threadIdx.x; j < kpb; j += NT) {
        const uint32_t key = (bin << shift) + j;
        const uint32_t r = key / D.T;
        S->rank[j] = r; S->step[j] = D.step_base + (key - r * D.T);
      }
    }
    uint4 pk[EPT];
    uint32_t where[EPT];
#pragma unroll
    for (uint32_t j = 0; j < EPT; ++j) {
      const uint32_t i = j * NT + threadIdx.x;
      where[j] = 0xFFFFFFFFu;
      pk[j] = nx[j];
      if (i < m) {
        const uint32_t kib = pk[j].x >> 19;
        where[j] = (kib << 16) | atomicAdd(&S->cnt[kib], 1u);
      }
    }
    if (tile + gridDim.x < n_tiles) {
      locate(tile + gridDim.x, nbin, ns0, nm);
#pragma unroll
      for (uint32_t j = 0; j < EPT; ++j) {
        const uint32_t i = j * NT + threadIdx.x;
        if (i < nm) nx[j] = ldcs128(coarse + (size_t)ns0 + i);
      }
    }
    __syncthreads();
    uint32_t c, pre;
    p2_bins_scan(S, c, pre);
    if (threadIdx.x < P2_MAX_BINS) {
      const uint32_t key = (bin << shift) + threadIdx.x;
      S->gbase[threadIdx.x] = ((c && key < RT) ? atomicAdd(&kcur[key], c) : 0u) - pre;
    }
    __syncthreads();
#pragma unroll
    for (uint32_t j = 0; j < EPT; ++j) {
      if (where[j] != 0xFFFFFFFFu) {
        const uint32_t kib = where[j] >> 16, slot = S->off[kib] + (where[j] & 0xFFFFu);
        const uint4 p = pk[j];
        // start + duration: 64-bit add
        const unsigned long long st = ((unsigned long long)p.w << 32) | p.z, en = st + p.y;
        sorted[2u * slot] = make_uint4(S->rank[kib], S->step[kib], p.x & 0x1FFFu, ((p.x >> 13) & 0x3Fu) << 16);
        sorted[2u * slot + 1u] = make_uint4(p.z, p.w, (uint32_t)en, (uint32_t)(en >> 32));
        S->binof[slot] = (uint8_t)kib;
      }
    }
    __syncthreads();
    // copy out, two threads per event: whole 32-byte sectors, consecutive inside every key's run
    for (uint32_t i = threadIdx.x; i < 2u * m; i += NT) {
      const uint32_t slot = i >> 1;
      grouped[2u * ((size_t)S->gbase[S->binof[slot]] + slot) + (i & 1u)] = sorted[i];
    }
    __syncthreads();
  }
}

// the slots behind the grouped events: invalid records (rank out of range), counted by the segmented kernel
__global__ void __launch_bounds__(256)
p2_pad_kernel(uint4* __restrict__ grouped, uint64_t n, const P2Small* __restrict__ sm) {
  const uint64_t stride = (uint64_t)gridDim.x * blockDim.x;
  for (uint64_t i = sm->n_valid + (uint64_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += stride) {
    grouped[2 * i] = make_uint4(0xFFFFFFFFu, 0xFFFFFFFFu, 0u, 0u);
    grouped[2 * i + 1] = make_uint4(0u, 0u, 0u, 0u);
  }
}

}  // namespace

// CTAs of the grouping pass and whether their key histograms (R*T + 1 counters) fit shared memory.
void argus_partition_plan(const argus_config* cfg, int sm_count, int max_smem_optin, uint32_t* n_cta,
                          bool* smem) {
  const size_t bin_bytes = sizeof(uint32_t) * ((size_t)cfg->n_ranks * cfg->n_steps + 1u);
  *smem = bin_bytes <= 200u * 1024u && bin_bytes + 1024u <= (size_t)max_smem_optin;
  *n_cta = *smem ? (uint32_t)sm_count * (bin_bytes <= 100u * 1024u ? 2u : 1u) : 0u;
}

// Two-level grouping: usable when the key counters (R*T) fit shared memory and sig / phase fit the packed word.
bool argus_partition2_plan(const argus_config* cfg, uint32_t* shift, size_t* small_bytes) {
  const uint64_t RT = (uint64_t)cfg->n_ranks * cfg->n_steps;
  if (RT > 24576u || cfg->n_sigs > 8192u || cfg->n_phases > 64u) return false;
  uint32_t bits = 0;
  while ((1ull << bits) < RT) ++bits;
  *shift = (bits + 1u) / 2u;                       // <= 8: at most 256 keys per bin, at most 256 bins
  *small_bytes = sizeof(P2Small);
  return true;
}

template <uint32_t NT, uint32_t EPT, int MINB>
static cudaError_t p2_coarse_go(argus_ctx* ctx, const uint4* src, uint64_t n, cudaStream_t s, bool configure) {
  const size_t smem = ((sizeof(P2SharedT<NT * EPT>) + 15u) & ~(size_t)15u) + (size_t)NT * EPT * 16u;
  if (configure)
    return cudaFuncSetAttribute(p2_coarse_kernel<NT, EPT, MINB>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
  p2_coarse_kernel<NT, EPT, MINB><<<(unsigned)ctx->sm_count * MINB, NT, smem, s>>>(
      src, n, ctx->dims, ctx->ws.part_shift, ctx->d_hist, reinterpret_cast<P2Small*>(ctx->d_part),
      reinterpret_cast<uint4*>(ctx->d_coarse), reinterpret_cast<uint4*>(ctx->d_group));
  return cudaGetLastError();
}
// coarse pass geometry: 256 threads x 4 events, three CTAs per SM.  Tiles of 512 events cost 20 % (128-byte
// runs per bin), 2,048-event tiles leave too few CTAs for the prefetched loads (register budget).
static cudaError_t p2_coarse_variant(argus_ctx* ctx, const uint4* src, uint64_t n, cudaStream_t s, bool configure) {
  return p2_coarse_go<256, 4, 3>(ctx, src, n, s, configure);
}

template <uint32_t NT, uint32_t EPT, int MINB>
static cudaError_t p2_fine_go(argus_ctx* ctx, const uint4* coarse, cudaStream_t s, bool configure, uint32_t* tile) {
  const size_t smem = ((sizeof(P2SharedT<NT * EPT>) + 15u) & ~(size_t)15u) + (size_t)NT * EPT * 32u;
  *tile = NT * EPT;
  if (configure)
    return cudaFuncSetAttribute(p2_fine_kernel<NT, EPT, MINB>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
  p2_fine_kernel<NT, EPT, MINB><<<(unsigned)ctx->sm_count * MINB, NT, smem, s>>>(
      coarse, ctx->dims, ctx->ws.part_shift, ctx->d_hist, reinterpret_cast<const P2Small*>(ctx->d_part),
      reinterpret_cast<uint4*>(ctx->d_group));
  return cudaGetLastError();
}
static uint32_t g_p2_tile = 1024u;            // tile of the fine pass (set by its configure call)
// fine pass geometry: 256 threads x 4 events, four CTAs per SM (64 registers hold the tile in hand and the
// prefetched one).  Geometries from 128 x 4 x 8 to 512 x 4 x 2 measured within 3 % once the loads are
// prefetched; without the prefetch the pass was 20 % slower at every geometry.
static cudaError_t p2_fine_variant(argus_ctx* ctx, const uint4* coarse, uint64_t, cudaStream_t s, bool configure) {
  return p2_fine_go<256, 4, 4>(ctx, coarse, s, configure, &g_p2_tile);
}

cudaError_t argus_configure_partition(argus_ctx* ctx) {
  if (ctx->ws.part_two_level) {
    const int cnt_bytes = (int)(sizeof(uint32_t) * ((size_t)ctx->dims.R * ctx->dims.T + P2_MAX_BINS));
    cudaError_t e = cudaFuncSetAttribute(p2_count_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, cnt_bytes);
    if (e == cudaSuccess) e = p2_coarse_variant(ctx, nullptr, 0, cudaStream_t(0), true);
    if (e == cudaSuccess) e = p2_fine_variant(ctx, nullptr, 0, cudaStream_t(0), true);
    return e;
  }
  if (!ctx->ws.part_smem) return cudaSuccess;
  const int bin_bytes = (int)(sizeof(uint32_t) * ((size_t)ctx->dims.R * ctx->dims.T + 1u));
  cudaError_t e = cudaFuncSetAttribute(partition_count_smem_kernel,
                                       cudaFuncAttributeMaxDynamicSharedMemorySize, bin_bytes);
  if (e == cudaSuccess)
    e = cudaFuncSetAttribute(partition_scatter_smem_kernel,
                             cudaFuncAttributeMaxDynamicSharedMemorySize, bin_bytes);
  return e;
}

// Group n <= cfg.max_ungrouped_events events by (rank, step) into the grouping area ctx->d_group.
cudaError_t argus_launch_partition(argus_ctx* ctx, const argus_event* ev, uint64_t n, cudaStream_t s) {
  const argus_dims& D = ctx->dims;
  const uint32_t m = D.R * D.T + 1u;
  const uint4* src = reinterpret_cast<const uint4*>(ev);
  const size_t bin_bytes = sizeof(uint32_t) * (size_t)m;
  if (ctx->ws.part_two_level) {
    const uint32_t RT = D.R * D.T, shift = ctx->ws.part_shift;
    P2Small* sm = reinterpret_cast<P2Small*>(ctx->d_part);
    uint4* coarse = reinterpret_cast<uint4*>(ctx->d_coarse);
    uint4* grouped = reinterpret_cast<uint4*>(ctx->d_group);
    cudaError_t e = cudaMemsetAsync(ctx->d_hist, 0, sizeof(uint32_t) * RT, s);
    if (e == cudaSuccess) e = cudaMemsetAsync(sm, 0, sizeof(P2Small), s);
    if (e != cudaSuccess) return e;
    const size_t cnt_bytes = sizeof(uint32_t) * ((size_t)RT + P2_MAX_BINS);
    uint32_t n_cta = (uint32_t)ctx->sm_count * (cnt_bytes <= 100u * 1024u ? 2u : 1u);
    uint64_t chunk = (n + n_cta - 1) / n_cta;
    chunk = (chunk + 1023) / 1024 * 1024;
    n_cta = (uint32_t)((n + chunk - 1) / chunk);
    p2_count_kernel<<<n_cta, 1024, cnt_bytes, s>>>(src, n, chunk, D, shift, ctx->d_hist, sm);
    p2_scan_kernel<<<1, 1024, 0, s>>>(ctx->d_hist, RT, sm, g_p2_tile);
    e = p2_coarse_variant(ctx, src, n, s, false);
    if (e != cudaSuccess) return e;
    e = p2_fine_variant(ctx, coarse, n, s, false);
    if (e != cudaSuccess) return e;
    p2_pad_kernel<<<(unsigned)ctx->sm_count * 4u, 256, 0, s>>>(grouped, n, sm);
    ctx->n_memsets += 2;
    ctx->n_kernels += 5;
    return cudaGetLastError();
  }
  if (ctx->ws.part_smem) {
    // per-CTA shared-memory histograms
    uint32_t n_cta = ctx->ws.part_ctas;
    uint64_t chunk = (n + n_cta - 1) / n_cta;
    chunk = (chunk + 1023) / 1024 * 1024;
    n_cta = (uint32_t)((n + chunk - 1) / chunk);
    uint32_t* H = ctx->d_part;
    partition_count_smem_kernel<<<n_cta, 1024, bin_bytes, s>>>(src, n, chunk, D, m, H);
    partition_offsets_kernel<<<(m + 255u) / 256u, 256, 0, s>>>(H, n_cta, m, ctx->d_hist);
    partition_scan_kernel<<<1, 1024, 0, s>>>(ctx->d_hist, m);
    partition_scatter_smem_kernel<<<n_cta, 1024, bin_bytes, s>>>(src, n, chunk, D, m, H, ctx->d_hist,
                                                                 reinterpret_cast<uint4*>(ctx->d_group));
    ctx->n_kernels += 4;
    return cudaGetLastError();
  }
  // too many groups for shared memory: one global counter array, L2 atomics
  cudaError_t e = cudaMemsetAsync(ctx->d_hist, 0, sizeof(uint32_t) * m, s);
  if (e != cudaSuccess) return e;
  uint64_t blocks = (n + 511) / 512;
  const uint64_t cap = (uint64_t)ctx->sm_count * 4 * 8;   // 4 CTAs of 512 per SM, a few tiles each
  if (blocks > cap) blocks = cap;
  partition_count_kernel<<<(unsigned)blocks, 512, 0, s>>>(src, n, D, ctx->d_hist);
  partition_scan_kernel<<<1, 1024, 0, s>>>(ctx->d_hist, m);
  partition_scatter_kernel<<<(unsigned)blocks, 512, 0, s>>>(src, n, D, ctx->d_hist,
                                                            reinterpret_cast<uint4*>(ctx->d_group));
  ctx->n_memsets += 1;
  ctx->n_kernels += 3;
  return cudaGetLastError();
}
