// diagnose.cu — cross-rank median/MAD selection kernel (NS (4): "per (step, sig), the exact median
// and MAD over ranks of the u64 summed duration and flags a rank when |x - median| > 3*MAD, all
// in integer arithmetic"; the paper's comparison of "the same kernel across different ranks",
// PAPER.md:228).  R15: the same rule runs on the phase spans and on the whole-iteration span.
//
// One CTA per series (step t, family member f: sig s < S, or span k = f - S <= P).  The R values
// live in registers (up to 16 per thread); order statistics come from an exact MSD radix select:
// a block min/max finds the highest bit in which the candidates differ, then 8-bit digit
// histograms in shared memory narrow the candidate set until one value remains.  No sort, no
// sampling, no floating point.
#include "argus_internal.cuh"

#include <mutex>

namespace {

constexpr int EPT = 16;
constexpr uint32_t FULL = 0xFFFFFFFFu;

struct SelSmem {
  uint32_t hist[256];
  unsigned long long red_a[32];
  unsigned long long red_b[32];
  unsigned long long bcast[2];
  uint32_t pick_digit, pick_before, pick_count;
};

template <typename K> __device__ __forceinline__ int top_bit(K v);     // index of the leading one (v != 0)
template <> __device__ __forceinline__ int top_bit<unsigned long long>(unsigned long long v) { return 63 - __clzll((long long)v); }
template <> __device__ __forceinline__ int top_bit<uint32_t>(uint32_t v) { return 31 - __clz((int)v); }

template <int NT, typename K>
__device__ __forceinline__ void block_minmax(K mn, K mx, SelSmem& sm, K& omn, K& omx) {
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) {
    K a = __shfl_xor_sync(FULL, mn, o), b = __shfl_xor_sync(FULL, mx, o);
    mn = a < mn ? a : mn;
    mx = b > mx ? b : mx;
  }
  const int w = threadIdx.x >> 5, lane = threadIdx.x & 31;
  __syncthreads();
  if (lane == 0) { sm.red_a[w] = mn; sm.red_b[w] = mx; }
  __syncthreads();
  mn = lane < NT / 32 ? (K)sm.red_a[lane] : (K)~(K)0;
  mx = lane < NT / 32 ? (K)sm.red_b[lane] : (K)0;
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) {
    K a = __shfl_xor_sync(FULL, mn, o), b = __shfl_xor_sync(FULL, mx, o);
    mn = a < mn ? a : mn;
    mx = b > mx ? b : mx;
  }
  omn = mn; omx = mx;
}

template <int NT>
__device__ __forceinline__ void block_sum2(uint32_t a, uint32_t b, SelSmem& sm, uint32_t& oa, uint32_t& ob) {
  a = __reduce_add_sync(FULL, a);
  b = __reduce_add_sync(FULL, b);
  const int w = threadIdx.x >> 5, lane = threadIdx.x & 31;
  __syncthreads();
  if (lane == 0) { sm.red_a[w] = a; sm.red_b[w] = b; }
  __syncthreads();
  a = lane < NT / 32 ? (uint32_t)sm.red_a[lane] : 0u;
  b = lane < NT / 32 ? (uint32_t)sm.red_b[lane] : 0u;
  oa = __reduce_add_sync(FULL, a);
  ob = __reduce_add_sync(FULL, b);
}

// k-th smallest (0-based) of the block's values v[j] (element index j*NT + tid < R).  Exact.
template <int NT, typename K>
__device__ K block_select(const K (&v)[EPT], uint32_t R, uint32_t k, SelSmem& sm) {
  const int tid = threadIdx.x;
  constexpr int TOP = (int)sizeof(K) * 8 - 1;
  K mn = (K)~(K)0, mx = (K)0;
#pragma unroll
  for (int j = 0; j < EPT; ++j)
    if ((uint32_t)(j * NT + tid) < R) { mn = v[j] < mn ? v[j] : mn; mx = v[j] > mx ? v[j] : mx; }
  block_minmax<NT, K>(mn, mx, sm, mn, mx);
  if (mn == mx) return mn;
  int top = top_bit<K>(mn ^ mx);                         // highest bit where candidates differ
  K prefix = (top == TOP) ? (K)0 : (K)((mn >> (top + 1)) << (top + 1));
  K pmask = (top == TOP) ? (K)0 : (K)(~(K)0 << (top + 1));   // bits already fixed
  int hi_bit = top;
  for (;;) {
    const int shift = hi_bit >= 7 ? hi_bit - 7 : 0;
    const uint32_t dmask = (1u << (hi_bit - shift + 1)) - 1u;
    __syncthreads();
    sm.hist[tid & 255] = 0u;
    if (NT < 256) for (int i = tid; i < 256; i += NT) sm.hist[i] = 0u;
    __syncthreads();
#pragma unroll
    for (int j = 0; j < EPT; ++j)
      if ((uint32_t)(j * NT + tid) < R && (v[j] & pmask) == prefix)
        atomicAdd(&sm.hist[(uint32_t)(v[j] >> shift) & dmask], 1u);
    __syncthreads();
    if (tid < 32) {
      // warp 0: 8 bins per lane, inclusive scan across lanes, pick the bin holding rank k
      uint32_t c[8], s = 0;
#pragma unroll
      for (int i = 0; i < 8; ++i) { c[i] = sm.hist[tid * 8 + i]; s += c[i]; }
      uint32_t inc = s;
#pragma unroll
      for (int o = 1; o < 32; o <<= 1) {
        uint32_t t = __shfl_up_sync(FULL, inc, o);
        if (tid >= o) inc += t;
      }
      uint32_t before = inc - s;
      if (k >= before && k < inc) {
#pragma unroll
        for (int i = 0; i < 8; ++i) {
          if (k >= before && k < before + c[i]) {
            sm.pick_digit = tid * 8 + i; sm.pick_before = before; sm.pick_count = c[i];
          }
          before += c[i];
        }
      }
    }
    __syncthreads();
    const uint32_t digit = sm.pick_digit, cnt = sm.pick_count;
    k -= sm.pick_before;
    prefix |= (K)digit << shift;
    pmask |= (K)dmask << shift;
    if (shift == 0) return prefix;
    if (cnt == 1u) {
      // a single candidate is left: whoever holds it publishes it
#pragma unroll
      for (int j = 0; j < EPT; ++j)
        if ((uint32_t)(j * NT + tid) < R && (v[j] & pmask) == prefix) sm.bcast[0] = v[j];
      __syncthreads();
      return (K)sm.bcast[0];
    }
    hi_bit = shift - 1;
  }
}

// median (R10) of the block's values: lo = v_(k), hi = v_(k+1 if R even), med = lo + (hi-lo)/2
template <int NT, typename K>
__device__ K block_median(const K (&v)[EPT], uint32_t R, SelSmem& sm) {
  const int tid = threadIdx.x;
  const uint32_t k = (R - 1) / 2;
  const K lo = block_select<NT, K>(v, R, k, sm);
  if ((R & 1u) != 0u) return lo;
  // hi = v[R/2] = v[k+1]: equals lo when at least k+2 values are <= lo, else the smallest value > lo
  uint32_t le = 0;
  K gt_min = (K)~(K)0;
#pragma unroll
  for (int j = 0; j < EPT; ++j)
    if ((uint32_t)(j * NT + tid) < R) {
      if (v[j] <= lo) ++le;
      else gt_min = v[j] < gt_min ? v[j] : gt_min;
    }
  uint32_t le_all, dummy;
  block_sum2<NT>(le, 0u, sm, le_all, dummy);
  K mn, mx;
  block_minmax<NT, K>(gt_min, (K)0, sm, mn, mx);
  const K hi = (le_all >= k + 2u) ? lo : mn;
  return lo + (hi - lo) / (K)2;
}

// K = uint32_t: the fast pass.  A series whose values span less than 2^32 (the usual case: per-rank
// sums of one kernel differ by far less than 4.29 s) is selected on exact 32-bit offsets from its
// minimum — half the registers, twice the resident CTAs; |x - med| fits 32 bits too.  A wider series is
// only marked in todo[].  K = unsigned long long: the second pass, which does the marked series.
// Where the series come from: the record table (and, for the sig series of the ctx's own table, its sum
// plane), or rank-contiguous planes handed in by the caller (argus_diagnose_planes: the exchanged
// planes of a rank-sharded job).
struct DiagSrc {
  const uint8_t* records;
  const unsigned long long* sig_plane;    // [T][S][rank_stride] or null
  const unsigned long long* span_plane;   // [T][P+1][rank_stride] or null
  uint32_t rank_stride;
  bool use_sums;
};

template <int NT, typename K>
__device__ __forceinline__ void diagnose_series(const DiagSrc& src, const argus_dims& D, const argus_diag_out& out,
                                                uint8_t* __restrict__ todo, uint32_t series_id, SelSmem& sm) {
  const uint8_t* __restrict__ records = src.records;
  const bool use_sums = src.use_sums;
  const int tid = threadIdx.x;
  const uint32_t F = D.S + D.P + 1u;
  const uint32_t t = series_id / F, f = series_id % F;
  const bool is_sig = f < D.S;
  const uint32_t R = D.R;
  if (is_sig ? (out.sig_stats == nullptr && out.sig_flags == nullptr && out.rank_score == nullptr)
             : (out.span_stats == nullptr && out.span_flags == nullptr && out.step_anomalous == nullptr))
    return;
  const unsigned long long* plane = is_sig ? src.sig_plane : src.span_plane;
  if (records == nullptr && plane == nullptr) return;      // planes mode without this family

  // ---- gather x[r] over ranks (a6) ----------------------------------------------------------
  unsigned long long x[EPT];
  const size_t off = is_sig ? (size_t)D.cell_off + (size_t)f * sizeof(argus_cell)
                            : (size_t)D.span_off + (size_t)(f - D.S) * sizeof(argus_span) + 16u;
#pragma unroll
  for (int j = 0; j < EPT; ++j) {
    const uint32_t r = (uint32_t)(j * NT + tid);
    x[j] = 0ull;
    if (r < R) {
      if (plane) {
        // rank-contiguous plane: one coalesced read per warp
        x[j] = __ldg(plane + ((size_t)t * (is_sig ? D.S : D.P + 1u) + (is_sig ? f : f - D.S)) * src.rank_stride + r);
      } else if (is_sig && use_sums) {
        // the sum plane: 8 bytes per rank, neighbouring sigs (other CTAs) share the sector
        x[j] = __ldg(D.sums + ((size_t)r * D.T + t) * D.S + f);
      } else {
        const ulonglong2 q = __ldg(reinterpret_cast<const ulonglong2*>(
            records + ((size_t)r * D.T + t) * D.rec_bytes + off));
        // cell: {count, sum} -> sum if count (R11: empty = 0);  span: {span_ns, n_events} -> span_ns
        x[j] = is_sig ? (q.x ? q.y : 0ull) : q.x;
      }
    }
  }
  // ---- a7 median, a8 MAD ----------------------------------------------------------------------
  K v[EPT];
  unsigned long long base = 0ull;
  if (sizeof(K) == 4) {
    unsigned long long xmn = ~0ull, xmx = 0ull;
#pragma unroll
    for (int j = 0; j < EPT; ++j)
      if ((uint32_t)(j * NT + tid) < R) { xmn = x[j] < xmn ? x[j] : xmn; xmx = x[j] > xmx ? x[j] : xmx; }
    block_minmax<NT, unsigned long long>(xmn, xmx, sm, xmn, xmx);
    const bool wide = xmx - xmn > 0xFFFFFFFFull;
    if (tid == 0) todo[series_id] = wide ? 1 : 0;
    if (wide) return;
    base = xmn;
  }
#pragma unroll
  for (int j = 0; j < EPT; ++j) v[j] = (uint32_t)(j * NT + tid) < R ? (K)(x[j] - base) : (K)0;
  const K med_k = block_median<NT, K>(v, R, sm);
  K dev[EPT];
#pragma unroll
  for (int j = 0; j < EPT; ++j) dev[j] = v[j] >= med_k ? v[j] - med_k : med_k - v[j];
  const K mad_k = block_median<NT, K>(dev, R, sm);
  const unsigned long long med = base + med_k, mad = mad_k;
  const unsigned long long thr = mad > 0xFFFFFFFFFFFFFFFFull / 3ull ? 0xFFFFFFFFFFFFFFFFull : 3ull * mad;  // R12
  // ---- flags + roll-ups -------------------------------------------------------------------------
  uint8_t* fl = is_sig ? out.sig_flags : out.span_flags;
  const size_t series = is_sig ? (size_t)t * D.S + f : (size_t)t * (D.P + 1u) + (f - D.S);
  uint32_t nh = 0, nl = 0;
#pragma unroll
  for (int j = 0; j < EPT; ++j) {
    const uint32_t r = (uint32_t)(j * NT + tid);
    if (r < R) {
      uint8_t g = ARGUS_FLAG_NONE;
      if ((unsigned long long)dev[j] > thr) g = v[j] > med_k ? ARGUS_FLAG_HIGH : ARGUS_FLAG_LOW;   // R13, R14
      nh += g == ARGUS_FLAG_HIGH;
      nl += g == ARGUS_FLAG_LOW;
      if (fl) fl[series * R + r] = g;
      if (is_sig && out.rank_score && g == ARGUS_FLAG_HIGH) atomicAdd(&out.rank_score[(size_t)t * R + r], 1u);
    }
  }
  uint32_t NH, NL;
  block_sum2<NT>(nh, nl, sm, NH, NL);
  if (tid == 0) {
    argus_series_stat st;
    st.median = med; st.mad = mad; st.n_high = NH; st.n_low = NL; st.reserved = 0;
    if (is_sig) { if (out.sig_stats) out.sig_stats[series] = st; }
    else {
      if (out.span_stats) out.span_stats[series] = st;
      if (f - D.S == D.P && out.step_anomalous) out.step_anomalous[t] = NH;
    }
  }
}

template <int NT, typename K>
__global__ void __launch_bounds__(NT, (sizeof(K) == 4 && NT <= 256) ? 1024 / NT : 1)
diagnose_kernel(DiagSrc src, argus_dims D, argus_diag_out out, uint8_t* __restrict__ todo, uint32_t n_series) {
  __shared__ SelSmem sm;
  if (sizeof(K) == 4) {                    // one CTA per series
    if (blockIdx.x < n_series) diagnose_series<NT, K>(src, D, out, todo, blockIdx.x, sm);
    return;
  }
  // K = 64 bit: a few CTAs, each scanning its share of the marks NT at a time (coalesced byte loads, so that
  // the usual case — no series spans 2^32 — costs one pass over the marks) and selecting the marked series
  __shared__ uint32_t s_list[NT];
  __shared__ uint32_t s_n;
  const uint32_t chunk = (n_series + gridDim.x - 1u) / gridDim.x;
  const uint32_t b0 = blockIdx.x * chunk, b1 = b0 + chunk < n_series ? b0 + chunk : n_series;
  for (uint32_t base = b0; base < b1; base += NT) {
    if (threadIdx.x == 0) s_n = 0u;
    __syncthreads();
    const uint32_t b = base + threadIdx.x;
    if (b < b1 && todo[b]) s_list[atomicAdd(&s_n, 1u)] = b;
    __syncthreads();
    const uint32_t cnt = s_n;
    for (uint32_t i = 0; i < cnt; ++i) {
      diagnose_series<NT, K>(src, D, out, todo, s_list[i], sm);
      __syncthreads();                     // the next series reuses sm
    }
  }
}

// ---- R <= 256: one WARP per series -----------------------------------------------------------------
// The block kernel above spends its time in block barriers (about ten radix passes of three barriers
// per selection, two selections per series) while a series of a few hundred ranks is 8 values per
// lane: here each warp owns a series, its digit histogram sits in 1 KB of shared memory of its own,
// and the only synchronisation is __syncwarp.  Series whose values span 2^32 or more are marked for the
// 64-bit pass (as in the block kernel).
template <int VPL>
__device__ __forceinline__ uint32_t warp_select(const uint32_t (&v)[VPL], uint32_t R, uint32_t k, uint32_t* hist) {
  const int lane = threadIdx.x & 31;
  uint32_t mn = 0xFFFFFFFFu, mx = 0u;
#pragma unroll
  for (int j = 0; j < VPL; ++j)
    if ((uint32_t)(j * 32 + lane) < R) { mn = v[j] < mn ? v[j] : mn; mx = v[j] > mx ? v[j] : mx; }
  mn = __reduce_min_sync(FULL, mn);
  mx = __reduce_max_sync(FULL, mx);
  if (mn == mx) return mn;
  const int top = 31 - __clz((int)(mn ^ mx));
  uint32_t prefix = top == 31 ? 0u : ((mn >> (top + 1)) << (top + 1));
  uint32_t pmask = top == 31 ? 0u : (0xFFFFFFFFu << (top + 1));
  int hi_bit = top;
  for (;;) {
    const int shift = hi_bit >= 7 ? hi_bit - 7 : 0;
    const uint32_t dmask = (1u << (hi_bit - shift + 1)) - 1u;
    __syncwarp();
#pragma unroll
    for (int i = 0; i < 8; ++i) hist[lane * 8 + i] = 0u;
    __syncwarp();
#pragma unroll
    for (int j = 0; j < VPL; ++j)
      if ((uint32_t)(j * 32 + lane) < R && (v[j] & pmask) == prefix) atomicAdd(&hist[(v[j] >> shift) & dmask], 1u);
    __syncwarp();
    uint32_t c[8], sum = 0;
#pragma unroll
    for (int i = 0; i < 8; ++i) { c[i] = hist[lane * 8 + i]; sum += c[i]; }
    uint32_t inc = sum;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
      const uint32_t t = __shfl_up_sync(FULL, inc, o);
      if (lane >= o) inc += t;
    }
    uint32_t before = inc - sum;
    const bool here = k >= before && k < inc;          // exactly one lane
    uint32_t digit = 0, dbefore = 0, dcount = 0;
    if (here) {
#pragma unroll
      for (int i = 0; i < 8; ++i) {
        if (k >= before && k < before + c[i]) { digit = (uint32_t)(lane * 8 + i); dbefore = before; dcount = c[i]; }
        before += c[i];
      }
    }
    const int src = __ffs((int)__ballot_sync(FULL, here)) - 1;
    digit = __shfl_sync(FULL, digit, src);
    dbefore = __shfl_sync(FULL, dbefore, src);
    dcount = __shfl_sync(FULL, dcount, src);
    k -= dbefore;
    prefix |= digit << shift;
    pmask |= dmask << shift;
    if (shift == 0) return prefix;
    if (dcount == 1u) {
      uint32_t val = 0;
      bool mine = false;
#pragma unroll
      for (int j = 0; j < VPL; ++j)
        if ((uint32_t)(j * 32 + lane) < R && (v[j] & pmask) == prefix) { val = v[j]; mine = true; }
      return __shfl_sync(FULL, val, __ffs((int)__ballot_sync(FULL, mine)) - 1);
    }
    hi_bit = shift - 1;
  }
}

template <int VPL>
__device__ __forceinline__ uint32_t warp_median(const uint32_t (&v)[VPL], uint32_t R, uint32_t* hist) {
  const int lane = threadIdx.x & 31;
  const uint32_t k = (R - 1) / 2;
  const uint32_t lo = warp_select<VPL>(v, R, k, hist);
  if (R & 1u) return lo;
  uint32_t le = 0, gt_min = 0xFFFFFFFFu;
#pragma unroll
  for (int j = 0; j < VPL; ++j)
    if ((uint32_t)(j * 32 + lane) < R) {
      if (v[j] <= lo) ++le;
      else gt_min = v[j] < gt_min ? v[j] : gt_min;
    }
  le = __reduce_add_sync(FULL, le);
  gt_min = __reduce_min_sync(FULL, gt_min);
  const uint32_t hi = le >= k + 2u ? lo : gt_min;     // R10: hi = v[R/2]
  return lo + (hi - lo) / 2u;
}

// WPC warps per CTA.  The kernel is a chain of dependent warp-wide steps per series (latency, not bandwidth):
// what helps is more resident warps.  R <= 256 keeps 8 values per lane, fits 56 registers and runs 9 CTAs of 4
// warps per SM, so that the 5,210 series of `mid` are ONE wave of 148 x 36 warps instead of one and a half.
template <int VPL, int WPC, int MINB>
__global__ void __launch_bounds__(WPC * 32, MINB)
diagnose_warp_kernel(DiagSrc src, argus_dims D, argus_diag_out out, uint8_t* __restrict__ todo, uint32_t n_series) {
  __shared__ uint32_t s_hist[WPC][256];
  const int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
  const uint32_t series_id = blockIdx.x * (uint32_t)WPC + (uint32_t)w;
  if (series_id >= n_series) return;
  uint32_t* hist = s_hist[w];
  const uint32_t F = D.S + D.P + 1u;
  const uint32_t t = series_id / F, f = series_id % F;
  const bool is_sig = f < D.S;
  const uint32_t R = D.R;
  if (lane == 0) todo[series_id] = 0;
  if (is_sig ? (out.sig_stats == nullptr && out.sig_flags == nullptr && out.rank_score == nullptr)
             : (out.span_stats == nullptr && out.span_flags == nullptr && out.step_anomalous == nullptr))
    return;
  const unsigned long long* plane = is_sig ? src.sig_plane : src.span_plane;
  if (src.records == nullptr && plane == nullptr) return;
  // ---- gather (a6) ------------------------------------------------------------------------------------
  unsigned long long x[VPL];
  const size_t off = is_sig ? (size_t)D.cell_off + (size_t)f * sizeof(argus_cell)
                            : (size_t)D.span_off + (size_t)(f - D.S) * sizeof(argus_span) + 16u;
  unsigned long long xmn = ~0ull, xmx = 0ull;
#pragma unroll
  for (int j = 0; j < VPL; ++j) {
    const uint32_t r = (uint32_t)(j * 32 + lane);
    x[j] = 0ull;
    if (r < R) {
      if (plane) {
        x[j] = __ldg(plane + ((size_t)t * (is_sig ? D.S : D.P + 1u) + (is_sig ? f : f - D.S)) * src.rank_stride + r);
      } else if (is_sig && src.use_sums) {
        x[j] = __ldg(D.sums + ((size_t)r * D.T + t) * D.S + f);
      } else {
        const ulonglong2 q = __ldg(reinterpret_cast<const ulonglong2*>(
            src.records + ((size_t)r * D.T + t) * D.rec_bytes + off));
        x[j] = is_sig ? (q.x ? q.y : 0ull) : q.x;
      }
      xmn = x[j] < xmn ? x[j] : xmn;
      xmx = x[j] > xmx ? x[j] : xmx;
    }
  }
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) {
    const unsigned long long a = __shfl_xor_sync(FULL, xmn, o), b = __shfl_xor_sync(FULL, xmx, o);
    xmn = a < xmn ? a : xmn;
    xmx = b > xmx ? b : xmx;
  }
  if (xmx - xmn > 0xFFFFFFFFull) {           // the 64-bit pass takes this series
    if (lane == 0) todo[series_id] = 1;
    return;
  }
  // ---- a7 median, a8 MAD on exact 32-bit offsets from the minimum ------------------------------------------
  uint32_t v[VPL], dev[VPL];
#pragma unroll
  for (int j = 0; j < VPL; ++j) v[j] = (uint32_t)(j * 32 + lane) < R ? (uint32_t)(x[j] - xmn) : 0u;
  const uint32_t med_k = warp_median<VPL>(v, R, hist);
#pragma unroll
  for (int j = 0; j < VPL; ++j) dev[j] = v[j] >= med_k ? v[j] - med_k : med_k - v[j];
  const uint32_t mad_k = warp_median<VPL>(dev, R, hist);
  const unsigned long long med = xmn + med_k, mad = mad_k;
  const unsigned long long thr = 3ull * mad;                         // mad < 2^32: no saturation (R12)
  // ---- flags + roll-ups ------------------------------------------------------------------------------------
  uint8_t* fl = is_sig ? out.sig_flags : out.span_flags;
  const size_t series = is_sig ? (size_t)t * D.S + f : (size_t)t * (D.P + 1u) + (f - D.S);
  uint32_t nh = 0, nl = 0;
#pragma unroll
  for (int j = 0; j < VPL; ++j) {
    const uint32_t r = (uint32_t)(j * 32 + lane);
    if (r < R) {
      uint8_t g = ARGUS_FLAG_NONE;
      if ((unsigned long long)dev[j] > thr) g = v[j] > med_k ? ARGUS_FLAG_HIGH : ARGUS_FLAG_LOW;   // R13, R14
      nh += g == ARGUS_FLAG_HIGH;
      nl += g == ARGUS_FLAG_LOW;
      if (fl) fl[series * R + r] = g;
      if (is_sig && out.rank_score && g == ARGUS_FLAG_HIGH) atomicAdd(&out.rank_score[(size_t)t * R + r], 1u);
    }
  }
  nh = __reduce_add_sync(FULL, nh);
  nl = __reduce_add_sync(FULL, nl);
  if (lane == 0) {
    argus_series_stat st;
    st.median = med; st.mad = mad; st.n_high = nh; st.n_low = nl; st.reserved = 0;
    if (is_sig) { if (out.sig_stats) out.sig_stats[series] = st; }
    else {
      if (out.span_stats) out.span_stats[series] = st;
      if (f - D.S == D.P && out.step_anomalous) out.step_anomalous[t] = nh;
    }
  }
}

}  // namespace

static cudaError_t launch_select(argus_ctx* ctx, const DiagSrc& src, const argus_dims& D, const argus_diag_out* o,
                                 cudaStream_t s) {
  if (o->rank_score) {
    cudaError_t e = cudaMemsetAsync(o->rank_score, 0, (size_t)D.T * D.R * sizeof(uint32_t), s);
    if (e != cudaSuccess) return e;
    ctx->n_memsets += 1;
  }
  const uint64_t blocks = (uint64_t)D.T * (D.S + D.P + 1u);     // <= the ctx's own series count (checked by callers)
  uint8_t* todo = ctx->d_diag_todo;        // one mark byte per series (workspace)
  const unsigned nb = (unsigned)blocks;
  // 32-bit pass: one warp per series up to 256 ranks, one CTA of R / 16 threads per series beyond; then the few series
  // that span 2^32 or more (marked in todo) in 64 bits, by a handful of CTAs that walk the marks
  const unsigned wide_grid = nb < (unsigned)ctx->sm_count * 2u ? nb : (unsigned)ctx->sm_count * 2u;
  if (D.R <= 256u) {
    diagnose_warp_kernel<8, 4, 9><<<(nb + 3u) / 4u, 128, 0, s>>>(src, D, *o, todo, nb);
    diagnose_kernel<64, unsigned long long><<<wide_grid, 64, 0, s>>>(src, D, *o, todo, nb);
  } else if (D.R <= 64u * EPT) {
    // 257 .. 1024 ranks: two warps per series, 16 values per thread (R = 1024: 119 us for 8,260 series against
    // 286 us with a warp per series and 32 values per lane, 256 us with 256-thread CTAs)
    diagnose_kernel<64, uint32_t><<<nb, 64, 0, s>>>(src, D, *o, todo, nb);
    diagnose_kernel<64, unsigned long long><<<wide_grid, 64, 0, s>>>(src, D, *o, todo, nb);
  } else if (D.R <= 128u * EPT) {
    diagnose_kernel<128, uint32_t><<<nb, 128, 0, s>>>(src, D, *o, todo, nb);
    diagnose_kernel<128, unsigned long long><<<wide_grid, 128, 0, s>>>(src, D, *o, todo, nb);
  } else if (D.R <= 256u * EPT) {
    diagnose_kernel<256, uint32_t><<<nb, 256, 0, s>>>(src, D, *o, todo, nb);
    diagnose_kernel<256, unsigned long long><<<wide_grid, 256, 0, s>>>(src, D, *o, todo, nb);
  } else {
    diagnose_kernel<1024, uint32_t><<<nb, 1024, 0, s>>>(src, D, *o, todo, nb);
    diagnose_kernel<1024, unsigned long long><<<wide_grid, 1024, 0, s>>>(src, D, *o, todo, nb);
  }
  ctx->n_kernels += 2;
  return cudaGetLastError();
}

cudaError_t argus_launch_diagnose(argus_ctx* ctx, const void* d_records, const argus_diag_out* o,
                                  bool use_sums, cudaStream_t s) {
  DiagSrc src;
  src.records = static_cast<const uint8_t*>(d_records);
  src.sig_plane = nullptr; src.span_plane = nullptr; src.rank_stride = 0; src.use_sums = use_sums;
  return launch_select(ctx, src, ctx->dims, o, s);
}

// Series handed in as rank-contiguous planes (a slice of the sigs of a job of pl->n_ranks ranks).
cudaError_t argus_launch_diagnose_planes(argus_ctx* ctx, const argus_planes* pl, const argus_diag_out* o,
                                         cudaStream_t s) {
  DiagSrc src;
  src.records = nullptr;
  src.sig_plane = reinterpret_cast<const unsigned long long*>(pl->sig_sums);
  src.span_plane = reinterpret_cast<const unsigned long long*>(pl->span_ns);
  src.rank_stride = pl->rank_stride; src.use_sums = false;
  argus_dims D = ctx->dims;
  D.R = pl->n_ranks; D.S = pl->n_sigs; D.sums = nullptr;
  return launch_select(ctx, src, D, o, s);
}

// ---- plane export of a rank shard (the ONE exchange of a rank-sharded job) ---------------
namespace {

// dst[((t*ns + (s - s0)) * stride + off + r] = sums[(r*T + t)*S + s]: tiled transpose through shared memory,
// reads coalesced over sigs, writes coalesced over ranks (rows of R_local u64 — whole lines for a peer).
__global__ void __launch_bounds__(256)
pack_sig_plane_kernel(const unsigned long long* __restrict__ sums, argus_dims D, uint32_t s0, uint32_t ns,
                      unsigned long long* __restrict__ dst, uint32_t stride, uint32_t off) {
  __shared__ unsigned long long tile[32][33];
  const uint32_t sb = blockIdx.x * 32u, rb = blockIdx.y * 32u;
  const uint32_t tx = threadIdx.x & 31u, ty = threadIdx.x >> 5;      // 32 x 8
  // gridDim.z = min(T, 65535) (the grid's z limit): a CTA walks the steps z, z + gridDim.z, ...
  for (uint32_t t = blockIdx.z; t < D.T; t += gridDim.z) {
    for (uint32_t i = ty; i < 32u; i += 8u) {
      const uint32_t r = rb + i, sg = sb + tx;
      tile[i][tx] = (r < D.R && sg < ns) ? __ldg(sums + ((size_t)r * D.T + t) * D.S + s0 + sg) : 0ull;
    }
    __syncthreads();
    for (uint32_t i = ty; i < 32u; i += 8u) {
      const uint32_t sg = sb + i, r = rb + tx;
      if (sg < ns && r < D.R) dst[((size_t)t * ns + sg) * stride + off + r] = tile[tx][i];
    }
    __syncthreads();                                                 // the next step reuses the tile
  }
}

// dst[((t*(P+1) + k) * stride + off + r] = span[r][t][k].span_ns of the finalised records
__global__ void __launch_bounds__(256)
pack_span_plane_kernel(const uint8_t* __restrict__ records, argus_dims D, unsigned long long* __restrict__ dst,
                       uint32_t stride, uint32_t off) {
  const uint64_t n = (uint64_t)D.T * (D.P + 1u) * D.R;                // R*T < 2^31, P <= 64: up to 2^37
  for (uint64_t i = (uint64_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (uint64_t)gridDim.x * blockDim.x) {
    const uint32_t r = (uint32_t)(i % D.R), tk = (uint32_t)(i / D.R), k = tk % (D.P + 1u), t = tk / (D.P + 1u);
    const argus_span* sp = reinterpret_cast<const argus_span*>(records + ((size_t)r * D.T + t) * D.rec_bytes + D.span_off) + k;
    dst[(size_t)tk * stride + off + r] = sp->span_ns;
  }
}

}  // namespace

cudaError_t argus_launch_pack_planes(argus_ctx* ctx, const void* d_records, uint32_t s0, uint32_t s1,
                                     uint64_t* dst_sig, uint64_t* dst_span, uint32_t stride, uint32_t off,
                                     cudaStream_t s) {
  const argus_dims& D = ctx->dims;
  if (dst_sig && s1 > s0) {
    const uint32_t ns = s1 - s0;
    dim3 grid((ns + 31u) / 32u, (D.R + 31u) / 32u, D.T < 65535u ? D.T : 65535u);
    pack_sig_plane_kernel<<<grid, 256, 0, s>>>(D.sums, D, s0, ns, reinterpret_cast<unsigned long long*>(dst_sig),
                                               stride, off);
    ctx->n_kernels += 1;
  }
  if (dst_span) {
    const uint64_t n = (uint64_t)D.T * (D.P + 1u) * D.R;
    const uint64_t want = (n + 255u) / 256u;                         // grid-stride beyond 2^20 CTAs
    pack_span_plane_kernel<<<(unsigned)(want < (1u << 20) ? want : (1u << 20)), 256, 0, s>>>(static_cast<const uint8_t*>(d_records), D,
                                                            reinterpret_cast<unsigned long long*>(dst_span), stride, off);
    ctx->n_kernels += 1;
  }
  return cudaGetLastError();
}

// ---- argus_diagnose_planes_static: the rule on planes for callers that may not allocate -------------------
// See include/argus.h for who needs this and why.  Everything the selection kernels touch beyond the caller's
// planes and outputs is the mark byte per series; here those bytes live in an array that is part of the
// library image, so the path has no ctx, no workspace and no allocation of any kind.
//
// g_static_marks is a DEVICE symbol.  In host code its name stands for a host-side shadow of the symbol, not for
// an address a kernel can use (a kernel handed &g_static_marks[0] from host code would fault, or scribble over
// host memory on a system where the GPU can reach it).  The address the kernels get comes from
// cudaGetSymbolAddress, asked once per device with that device current, and is cached below.
static __device__ __align__(256) uint8_t g_static_marks[ARGUS_STATIC_MAX_SERIES];

namespace {
struct StaticDevice {
  uint8_t* marks;     // device address of g_static_marks on this device (null: not looked up yet)
  int sm_count;
};
StaticDevice g_static_dev[ARGUS_STATIC_MAX_DEVICES];
std::mutex g_static_mu;

// First call on `dev` (which is current): symbol address + SM count.  Host-side queries only.
cudaError_t static_device(int dev, StaticDevice* out) {
  std::lock_guard<std::mutex> lock(g_static_mu);
  StaticDevice& d = g_static_dev[dev];
  if (d.marks == nullptr) {
    uint8_t* p = nullptr;
    cudaError_t e = cudaGetSymbolAddress(reinterpret_cast<void**>(&p), g_static_marks);
    if (e != cudaSuccess) return e;
    int sms = 0;
    e = cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
    if (e != cudaSuccess) return e;
    if (p == nullptr || sms <= 0) return cudaErrorInvalidSymbol;
    d.sm_count = sms;
    d.marks = p;
  }
  *out = d;
  return cudaSuccess;
}
}  // namespace

extern "C" int argus_diagnose_planes_static(const argus_planes* pl, uint32_t n_steps, uint32_t n_phases,
                                            const argus_diag_out* outs, void* stream) {
  if (!pl || !outs) return ARGUS_EINVAL;
  if (n_steps == 0 || n_phases == 0 || n_phases > ARGUS_MAX_PHASES) return ARGUS_EINVAL;
  if (pl->n_ranks == 0 || pl->n_ranks > ARGUS_MAX_RANKS || pl->rank_stride < pl->n_ranks) return ARGUS_EINVAL;
  if ((pl->n_sigs != 0) != (pl->sig_sums != nullptr)) return ARGUS_EINVAL;
  if (((uintptr_t)pl->sig_sums & 7u) || ((uintptr_t)pl->span_ns & 7u)) return ARGUS_EINVAL;
  if (((uintptr_t)outs->sig_stats & 15u) || ((uintptr_t)outs->span_stats & 15u)) return ARGUS_EINVAL;
  if (((uintptr_t)outs->rank_score & 3u) || ((uintptr_t)outs->step_anomalous & 3u)) return ARGUS_EINVAL;
  // the fixed array bounds the job: one mark byte per (step, sig or span) series
  const uint64_t n_series = (uint64_t)n_steps * ((uint64_t)pl->n_sigs + n_phases + 1u);
  if (n_series > ARGUS_STATIC_MAX_SERIES) return ARGUS_ESIZE;
  int dev = -1;
  if (cudaGetDevice(&dev) != cudaSuccess) return ARGUS_ECUDA;
  if (dev < 0 || dev >= ARGUS_STATIC_MAX_DEVICES) return ARGUS_EINVAL;
  StaticDevice sd;
  if (static_device(dev, &sd) != cudaSuccess) return ARGUS_ECUDA;
  cudaStream_t s = (cudaStream_t)stream;
  // The array keeps whatever the previous call (of any geometry) left in it: start from clean marks.
  if (cudaMemsetAsync(sd.marks, 0, (size_t)n_series, s) != cudaSuccess) return ARGUS_ECUDA;
  // launch_select reads three things of a ctx — where the marks are, the SM count, the launch counters —
  // so a stand-in on the stack carries them; nothing else of it is looked at in planes mode.
  argus_ctx tmp{};
  tmp.d_diag_todo = sd.marks;
  tmp.sm_count = sd.sm_count;
  DiagSrc src;
  src.records = nullptr;
  src.sig_plane = reinterpret_cast<const unsigned long long*>(pl->sig_sums);
  src.span_plane = reinterpret_cast<const unsigned long long*>(pl->span_ns);
  src.rank_stride = pl->rank_stride; src.use_sums = false;
  argus_dims D{};
  D.R = pl->n_ranks; D.T = n_steps; D.S = pl->n_sigs; D.P = n_phases; D.sums = nullptr;
  if (launch_select(&tmp, src, D, outs, s) != cudaSuccess) return ARGUS_ECUDA;
  return ARGUS_OK;
}
