// paper_literal.cu — the paper's own float algorithms on top of the integer path (SURVEY §8(f) NEXT-1..3):
//   NEXT-1  online statistical compression: log transform -> KDE on an equally spaced grid with Scott's
//           bandwidth (eq. 1) -> valleys -> two filters -> per-cluster (count, p50, p99)
//   NEXT-2  L3: log-normal mixture CDF (eq. 2) -> W1 by trapezoid on a log-uniform grid (eq. 3) -> mean-W1
//           deviation score -> IQR upper fence (eq. 4)
//   NEXT-3  L2: CV + z-score within a parallelism group (eq. 5, Table 3); L1: sliding-window ratio-gated
//           jitter detection and full-scan change point
// All in fp64 (the oracle's precision; where a float decides an integer — a valley, a flag — both sides
// decide in fp64).  Constants the paper leaves open are parameters; their defaults are the readings
// R23-R36 of DESIGN.md §3.  None of this is a contraction: no tensor cores.
#include <math.h>

#include "argus_internal.cuh"

namespace {

constexpr uint32_t FULL = 0xFFFFFFFFu;

// ---- NEXT-1: fine histogram ---------------------------------------------------------------------------
// R23: bin(d) = floor(8 log2 d) in [0, 255], decided in integers: b = floor(log2 d), m = d normalised to 32
// bits, sub = #{j in 1..7 : m >= ceil(2^(31 + j/8))} — exact because m is an integer and 2^(31 + j/8) is not.
__device__ __forceinline__ uint32_t fine_bin(unsigned long long d) {
  if (d <= 1ull) return 0u;
  if (d >> 32) return 255u;
  const uint32_t d32 = (uint32_t)d;
  const uint32_t b = 31u - (uint32_t)__clz((int)d32);
  const uint32_t m = d32 << (31u - b);
  const uint32_t sub = (m >= 0x8b95c1e4u) + (m >= 0x9837f052u) + (m >= 0xa5fed6aau) + (m >= 0xb504f334u) +
                       (m >= 0xc5672a12u) + (m >= 0xd744fccbu) + (m >= 0xeac0c6e8u);
  return 8u * b + sub;
}

__global__ void __launch_bounds__(256)
fine_hist_kernel(const uint4* __restrict__ ev, uint64_t n, argus_dims D, uint32_t* __restrict__ hist) {
  const uint64_t stride = (uint64_t)gridDim.x * blockDim.x;
  for (uint64_t i = (uint64_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += stride) {
    const uint4 lo = __ldcs(ev + 2 * i), hi = __ldcs(ev + 2 * i + 1);
    const long long start = (long long)(((unsigned long long)hi.y << 32) | hi.x);
    const long long end = (long long)(((unsigned long long)hi.w << 32) | hi.z);
    uint32_t key;
    if (!argus_event_key(D, lo.x, lo.y, lo.z, lo.w >> 16, start, end, key)) continue;
    atomicAdd(&hist[((size_t)key * D.S + lo.z) * 256u + fine_bin((unsigned long long)(end - start))], 1u);
  }
}

// ---- NEXT-1: KDE -> valleys -> filters -> triples, one warp per histogram ---------------------------------
constexpr int KDE_MAX_BINS = 256;
template <int NB>
struct KdeSmemT {
  double f[NB];
  double e[NB];                  // kernel weight by distance in grid steps
  uint32_t c[NB];
};
typedef KdeSmemT<KDE_MAX_BINS> KdeSmem;

// hist: n_bins counters of this cell (global, stride 1).  Lanes share the grid points; lane 0 walks the valleys.
template <class SM>
__device__ void kde_cell(const uint32_t* __restrict__ hist, const argus_kde_params& P, SM& sm,
                         argus_cluster* __restrict__ out, uint8_t* __restrict__ out_n, double* __restrict__ dens) {
  const int lane = threadIdx.x & 31;
  const uint32_t nb = P.n_bins;
  const double step = 0.6931471805599453 / (double)P.per_octave;     // ln 2 / bins per octave
  // counts, occupied range, n, mean
  double n = 0.0, sx = 0.0;
  uint32_t lo = nb, hi = 0;
  for (uint32_t b = lane; b < nb; b += 32) {
    const uint32_t c = hist[b];
    sm.c[b] = c;
    sm.f[b] = 0.0;
    if (c) {
      n += (double)c;
      sx += (double)c * (((double)b + 0.5) * step);
      lo = b < lo ? b : lo;
      hi = b > hi ? b : hi;
    }
  }
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) {
    n += __shfl_xor_sync(FULL, n, o);
    sx += __shfl_xor_sync(FULL, sx, o);
  }
  lo = __reduce_min_sync(FULL, lo);
  hi = __reduce_max_sync(FULL, hi);
  __syncwarp();
  for (uint32_t k = lane; k < P.max_clusters; k += 32) { out[k].count = 0u; out[k].p50_bin = 0; out[k].p99_bin = 0; }
  if (n == 0.0) {
    if (lane == 0) *out_n = 0;
    if (dens) for (uint32_t b = lane; b < nb; b += 32) dens[b] = 0.0;
    return;
  }
  double h = 0.0;
  if (n >= 2.0 && hi > lo) {            // R26: a single occupied bin (sigma = 0) has no density
    const double mean = sx / n;
    double ss = 0.0;
    for (uint32_t b = lo + lane; b <= hi; b += 32) {
      const double dx = ((double)b + 0.5) * step - mean;
      ss += (double)sm.c[b] * dx * dx;
    }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) ss += __shfl_xor_sync(FULL, ss, o);
    const double sigma = sqrt(ss / (n - 1.0));                        // R25: sample standard deviation (> 0: two bins)
    {
      h = 1.06 * sigma * pow(n, -0.2);                                // Scott's rule
      const double norm = 1.0 / (n * h * 2.5066282746310002);         // 1 / (n h sqrt(2 pi)): eq. (1), R22
      // the density is needed where valleys can lie: the occupied range (it is tabulated on the whole grid
      // only when the caller asks for it)
      // The grid is equally spaced, so the kernel weight of a (grid point, sample bin) pair depends on their
      // distance in grid steps only: tabulate K(d step / h) once per distance (hi - lo + 1 values of exp for
      // the occupied range instead of its square; sm.e) and sum with it, in bin order as before.
      const uint32_t j0 = dens ? 0u : lo, j1 = dens ? nb - 1u : hi;
      const uint32_t dmax = (j1 > hi ? j1 - lo : hi - lo) > (hi - j0) ? (j1 > hi ? j1 - lo : hi - lo) : (hi - j0);
      for (uint32_t d = lane; d <= dmax; d += 32) {
        const double u = ((double)d * step) / h;
        sm.e[d] = exp(-0.5 * u * u);
      }
      __syncwarp();
      for (uint32_t j = j0 + lane; j <= j1; j += 32) {
        double acc = 0.0;
        for (uint32_t b = lo; b <= hi; ++b) {
          const uint32_t c = sm.c[b];
          if (c) acc += (double)c * sm.e[j > b ? j - b : b - j];
        }
        sm.f[j] = acc * norm;
      }
    }
  }
  __syncwarp();
  if (dens) for (uint32_t b = lane; b < nb; b += 32) dens[b] = sm.f[b];
  if (lane == 0) {
    // valleys (R27), cluster-level filter (R28), spacing filter (R29); then the triples (R30)
    double need = P.min_frac * n;
    if ((double)P.min_count > need) need = (double)P.min_count;
    uint32_t n_out = 0;
    uint32_t seg_lo = lo;                   // first bin of the current cluster
    double since = 0.0, right = n;          // samples in [seg_lo, j), samples in [j, hi]
    uint32_t last_bound = 0;
    bool have_bound = false;
    auto emit = [&](uint32_t a, uint32_t b) {          // cluster of the bins [a, b)
      unsigned long long cnt = 0;
      for (uint32_t q = a; q < b; ++q) cnt += sm.c[q];
      if (cnt == 0ull || n_out >= P.max_clusters) return;
      const unsigned long long t50 = (cnt + 1ull) / 2ull;                     // ceil(0.5 cnt)
      const unsigned long long t99 = (unsigned long long)ceil(0.99 * (double)cnt);
      unsigned long long cum = 0;
      uint32_t p50 = b - 1u, p99 = b - 1u;
      bool got50 = false, got99 = false;
      for (uint32_t q = a; q < b; ++q) {
        cum += sm.c[q];
        if (!got50 && cum >= t50) { p50 = q; got50 = true; }
        if (!got99 && cum >= t99) { p99 = q; got99 = true; }
      }
      out[n_out].count = (uint32_t)cnt; out[n_out].p50_bin = (uint16_t)p50; out[n_out].p99_bin = (uint16_t)p99;
      ++n_out;
    };
    if (h > 0.0) {
      for (uint32_t j = lo + 1u; j < hi; ++j) {
        since += (double)sm.c[j - 1u];
        right -= (double)sm.c[j - 1u];
        if (sm.f[j] < sm.f[j - 1u] && sm.f[j] <= sm.f[j + 1u]) {
          const bool spaced = !have_bound || j - last_bound >= P.min_gap_bins;
          if (since >= need && right >= need && spaced && n_out + 1u < P.max_clusters) {   // the last slot takes the rest
            emit(seg_lo, j);
            seg_lo = j; since = 0.0; last_bound = j; have_bound = true;
          }
        }
      }
    }
    emit(seg_lo, hi + 1u);
    *out_n = (uint8_t)n_out;
  }
}

// The same algorithm with EIGHT lanes per histogram (four histograms per warp), for cells whose occupied bins span
// at most KDE_WIN grid steps (8 octaves on the fine grid: all but pathological cells).  A warp per cell leaves most
// lanes idle — the occupied range is a dozen bins — and the kernel is bound by instruction issue, so four cells per
// warp instruction is what counts.  Shared arrays are indexed relative to the first occupied bin.  Every formula
// and every decision is kde_cell's; only the order of the partial sums of the mean and the variance differs (8
// lanes instead of 32).  Returns false, having written nothing, when the cell is too wide.
template <uint32_t WIN>
struct KdeGrpT {
  static constexpr uint32_t win = WIN;
  double f[WIN];
  double e[WIN];
  uint32_t c[WIN];
};
typedef KdeGrpT<64> KdeGrp;

template <class GS>
__device__ bool kde_cell_group(const uint32_t* __restrict__ hist, const argus_kde_params& P, GS& sm,
                               argus_cluster* __restrict__ out, uint8_t* __restrict__ out_n) {
  constexpr uint32_t KDE_WIN = GS::win;
  const int lane = threadIdx.x & 31, gl = lane & 7;
  const uint32_t gmask = 0xFFu << (lane & 24);
  const uint32_t nb = P.n_bins;
  const double step = 0.6931471805599453 / (double)P.per_octave;
  // occupied range and n (integers: exact in any order)
  unsigned long long cnt = 0ull;
  uint32_t lo = nb, hi = 0;
  if ((nb & 3u) == 0u && (reinterpret_cast<size_t>(hist) & 15u) == 0u) {
    const uint4* h4 = reinterpret_cast<const uint4*>(hist);
    for (uint32_t q = gl; q < nb / 4u; q += 8) {
      const uint4 v = __ldg(h4 + q);
      const uint32_t w[4] = {v.x, v.y, v.z, v.w};
#pragma unroll
      for (uint32_t k = 0; k < 4u; ++k)
        if (w[k]) { const uint32_t b = 4u * q + k; cnt += w[k]; lo = b < lo ? b : lo; hi = b > hi ? b : hi; }
    }
  } else {
    for (uint32_t b = gl; b < nb; b += 8) {
      const uint32_t c = __ldg(hist + b);
      if (c) { cnt += c; lo = b < lo ? b : lo; hi = b > hi ? b : hi; }
    }
  }
#pragma unroll
  for (int o = 4; o > 0; o >>= 1) {
    cnt += __shfl_xor_sync(gmask, cnt, o);
    const uint32_t l2 = __shfl_xor_sync(gmask, lo, o), h2 = __shfl_xor_sync(gmask, hi, o);
    lo = l2 < lo ? l2 : lo; hi = h2 > hi ? h2 : hi;
  }
  if (cnt != 0ull && hi - lo >= KDE_WIN) return false;
  for (uint32_t k = gl; k < P.max_clusters; k += 8) { out[k].count = 0u; out[k].p50_bin = 0; out[k].p99_bin = 0; }
  if (cnt == 0ull) {
    if (gl == 0) *out_n = 0;
    return true;
  }
  const double n = (double)cnt;
  double sx = 0.0;
  for (uint32_t b = lo + gl; b <= hi; b += 8) {
    const uint32_t c = __ldg(hist + b);
    sm.c[b - lo] = c;
    sm.f[b - lo] = 0.0;
    if (c) sx += (double)c * (((double)b + 0.5) * step);
  }
#pragma unroll
  for (int o = 4; o > 0; o >>= 1) sx += __shfl_xor_sync(gmask, sx, o);
  __syncwarp(gmask);
  double h = 0.0;
  if (n >= 2.0 && hi > lo) {            // R26
    const double mean = sx / n;
    double ss = 0.0;
    for (uint32_t b = lo + gl; b <= hi; b += 8) {
      const double dx = ((double)b + 0.5) * step - mean;
      ss += (double)sm.c[b - lo] * dx * dx;
    }
#pragma unroll
    for (int o = 4; o > 0; o >>= 1) ss += __shfl_xor_sync(gmask, ss, o);
    const double sigma = sqrt(ss / (n - 1.0));                        // R25
    h = 1.06 * sigma * pow(n, -0.2);                                  // Scott's rule
    const double norm = 1.0 / (n * h * 2.5066282746310002);           // eq. (1), R22
    for (uint32_t d = gl; d <= hi - lo; d += 8) {
      const double u = ((double)d * step) / h;
      sm.e[d] = exp(-0.5 * u * u);
    }
    __syncwarp(gmask);
    for (uint32_t j = lo + gl; j <= hi; j += 8) {
      double acc = 0.0;
      for (uint32_t b = lo; b <= hi; ++b) {
        const uint32_t c = sm.c[b - lo];
        if (c) acc += (double)c * sm.e[j > b ? j - b : b - j];
      }
      sm.f[j - lo] = acc * norm;
    }
  }
  __syncwarp(gmask);
  if (gl == 0) {
    double need = P.min_frac * n;
    if ((double)P.min_count > need) need = (double)P.min_count;
    uint32_t n_out = 0;
    uint32_t seg_lo = lo;
    double since = 0.0, right = n;
    uint32_t last_bound = 0;
    bool have_bound = false;
    auto emit = [&](uint32_t a, uint32_t b) {          // cluster of the bins [a, b)
      unsigned long long cn = 0;
      for (uint32_t q = a; q < b; ++q) cn += sm.c[q - lo];
      if (cn == 0ull || n_out >= P.max_clusters) return;
      const unsigned long long t50 = (cn + 1ull) / 2ull;
      const unsigned long long t99 = (unsigned long long)ceil(0.99 * (double)cn);
      unsigned long long cum = 0;
      uint32_t p50 = b - 1u, p99 = b - 1u;
      bool got50 = false, got99 = false;
      for (uint32_t q = a; q < b; ++q) {
        cum += sm.c[q - lo];
        if (!got50 && cum >= t50) { p50 = q; got50 = true; }
        if (!got99 && cum >= t99) { p99 = q; got99 = true; }
      }
      out[n_out].count = (uint32_t)cn; out[n_out].p50_bin = (uint16_t)p50; out[n_out].p99_bin = (uint16_t)p99;
      ++n_out;
    };
    if (h > 0.0) {
      for (uint32_t j = lo + 1u; j < hi; ++j) {
        since += (double)sm.c[j - 1u - lo];
        right -= (double)sm.c[j - 1u - lo];
        if (sm.f[j - lo] < sm.f[j - 1u - lo] && sm.f[j - lo] <= sm.f[j + 1u - lo]) {
          const bool spaced = !have_bound || j - last_bound >= P.min_gap_bins;
          if (since >= need && right >= need && spaced && n_out + 1u < P.max_clusters) {
            emit(seg_lo, j);
            seg_lo = j; since = 0.0; last_bound = j; have_bound = true;
          }
        }
      }
    }
    emit(seg_lo, hi + 1u);
    *out_n = (uint8_t)n_out;
  }
  __syncwarp(gmask);
  return true;
}

// 32 cells per CTA: eight lanes each; the cells that are too wide for the group path — and every cell when the
// caller wants the density on the whole grid — are queued and take the warp path in the second half.
__global__ void __launch_bounds__(256)
kde_hist_kernel(const uint32_t* __restrict__ hist, uint64_t n_cells, argus_kde_params P, argus_cluster* clusters,
                uint8_t* n_clusters, double* density) {
  __shared__ union { KdeGrp g[32]; KdeSmem w[8]; } sm;
  __shared__ uint32_t s_wide[32];
  __shared__ uint32_t s_nwide;
  const uint64_t cell0 = (uint64_t)blockIdx.x * 32u;
  const uint32_t grp = threadIdx.x >> 3;
  if (threadIdx.x == 0) s_nwide = 0u;
  __syncthreads();
  const uint64_t cell = cell0 + grp;
  if (cell < n_cells) {
    bool done = false;
    if (density == nullptr)
      done = kde_cell_group(hist + cell * P.n_bins, P, sm.g[grp], clusters + cell * P.max_clusters, n_clusters + cell);
    if (!done && (threadIdx.x & 7) == 0) s_wide[atomicAdd(&s_nwide, 1u)] = grp;
  }
  __syncthreads();
  const uint32_t n_wide = s_nwide;
  for (uint32_t i = threadIdx.x >> 5; i < n_wide; i += 8) {
    const uint64_t wc = cell0 + s_wide[i];
    kde_cell(hist + wc * P.n_bins, P, sm.w[threadIdx.x >> 5], clusters + wc * P.max_clusters, n_clusters + wc,
             density ? density + wc * P.n_bins : nullptr);
    __syncwarp();
  }
}

// The 32-bucket histograms of the finalised record table (per_octave = 1, n_bins = 32).  A valley needs a bin
// strictly inside the occupied range (R27): a cell whose occupied buckets span fewer than three (nearly every
// cell: the compact cells of the aggregation hold four buckets at most, and 10 % jitter fills one or two) is ONE
// cluster whatever its density looks like, and its (count, p50, p99) are integer work — one thread does it,
// no floating point but the ceil(0.99 count) the wide path takes too.  The other cells are queued in shared
// memory and get the full KDE, eight lanes each (kde_cell_group), in the second half of the kernel.
constexpr int KDE_REC_NT = 256;
__global__ void __launch_bounds__(KDE_REC_NT)
kde_records_kernel(const uint8_t* __restrict__ records, argus_dims D, argus_kde_params P, argus_cluster* clusters,
                   uint8_t* n_clusters) {
  __shared__ KdeGrpT<32> sm[KDE_REC_NT / 8];
  __shared__ uint32_t s_wide[KDE_REC_NT];
  __shared__ uint32_t s_nwide;
  const uint64_t n_cells = (uint64_t)D.R * D.T * D.S;
  const uint64_t cell0 = (uint64_t)blockIdx.x * KDE_REC_NT;
  if (threadIdx.x == 0) s_nwide = 0u;
  __syncthreads();
  const uint64_t cell = cell0 + threadIdx.x;
  if (cell < n_cells) {
    const uint64_t rec = cell / D.S;
    const uint32_t sig = (uint32_t)(cell - rec * D.S);
    const argus_cell* c = reinterpret_cast<const argus_cell*>(records + rec * D.rec_bytes + D.cell_off) + sig;
    const uint4* h4 = reinterpret_cast<const uint4*>(c->hist);
    uint32_t lo = 32u, hi = 0u;
    unsigned long long n = 0ull;
#pragma unroll
    for (uint32_t q = 0; q < 8u; ++q) {
      const uint4 v = __ldg(h4 + q);
      const uint32_t w[4] = {v.x, v.y, v.z, v.w};
#pragma unroll
      for (uint32_t k = 0; k < 4u; ++k) {
        if (w[k]) {
          const uint32_t b = 4u * q + k;
          n += w[k];
          lo = b < lo ? b : lo;
          hi = b;
        }
      }
    }
    if (n != 0ull && hi - lo >= 2u) {
      s_wide[atomicAdd(&s_nwide, 1u)] = threadIdx.x;
    } else {
      argus_cluster* out = clusters + cell * P.max_clusters;
      argus_cluster first;
      first.count = 0u; first.p50_bin = 0; first.p99_bin = 0;
      if (n != 0ull) {
        const unsigned long long t50 = (n + 1ull) / 2ull, t99 = (unsigned long long)ceil(0.99 * (double)n);
        const unsigned long long c_lo = c->hist[lo];
        first.count = (uint32_t)n;
        first.p50_bin = (uint16_t)(c_lo >= t50 ? lo : hi);
        first.p99_bin = (uint16_t)(c_lo >= t99 ? lo : hi);
      }
      const uint32_t w1 = (uint32_t)first.p50_bin | ((uint32_t)first.p99_bin << 16);
      if ((P.max_clusters & 1u) == 0u) {           // slots of a cell are 16-byte aligned: whole-sector stores
        uint4* o4 = reinterpret_cast<uint4*>(out);
        o4[0] = make_uint4(first.count, w1, 0u, 0u);
        for (uint32_t k = 1; k < P.max_clusters / 2u; ++k) o4[k] = make_uint4(0u, 0u, 0u, 0u);
      } else {
        out[0] = first;
        argus_cluster z;
        z.count = 0u; z.p50_bin = 0; z.p99_bin = 0;
        for (uint32_t k = 1; k < P.max_clusters; ++k) out[k] = z;
      }
      n_clusters[cell] = n != 0ull ? 1 : 0;
    }
  }
  __syncthreads();
  const uint32_t n_wide = s_nwide;
  for (uint32_t i = threadIdx.x >> 3; i < n_wide; i += KDE_REC_NT / 8) {      // eight lanes per wide cell
    const uint64_t wc = cell0 + s_wide[i];
    const uint64_t rec = wc / D.S;
    const uint32_t sig = (uint32_t)(wc - rec * D.S);
    const argus_cell* c = reinterpret_cast<const argus_cell*>(records + rec * D.rec_bytes + D.cell_off) + sig;
    kde_cell_group(c->hist, P, sm[threadIdx.x >> 3], clusters + wc * P.max_clusters, n_clusters + wc);   // 32 bins: never too wide
  }
}

// clusters [R][T][S][mc] (rank-major, as argus_kde_clusters_records writes them) -> the L3 input
// [key = t*S + s][R][mc]: count, p50, p99 in ns (a bin stands for its geometric centre, R30)
__global__ void __launch_bounds__(256)
clusters_to_l3_kernel(const argus_cluster* __restrict__ cl, argus_dims D, uint32_t mc, uint32_t per_octave,
                      uint32_t* __restrict__ count, double* __restrict__ p50, double* __restrict__ p99) {
  // a bin stands for 2^((bin + 0.5) / per_octave) ns: 65,536 possible bins at most 256 of which a grid uses —
  // tabulate the first 256 with the very expression used for the others
  __shared__ double s_val[256];
  for (uint32_t b = threadIdx.x; b < 256u; b += blockDim.x) s_val[b] = exp2(((double)b + 0.5) / (double)per_octave);
  __syncthreads();
  const uint64_t n = (uint64_t)D.R * D.T * D.S * mc;
  for (uint64_t o = (uint64_t)blockIdx.x * blockDim.x + threadIdx.x; o < n; o += (uint64_t)gridDim.x * blockDim.x) {
    // o walks the OUTPUT (coalesced writes): o = ((key * R) + r) * mc + c
    const uint32_t c = (uint32_t)(o % mc);
    const uint64_t kr = o / mc;
    const uint32_t r = (uint32_t)(kr % D.R);
    const uint64_t key = kr / D.R;
    const argus_cluster q = cl[(((uint64_t)r * D.T * D.S) + key) * mc + c];
    count[o] = q.count;
    p50[o] = q.count ? (q.p50_bin < 256u ? s_val[q.p50_bin] : exp2(((double)q.p50_bin + 0.5) / (double)per_octave)) : 1.0;
    p99[o] = q.count ? (q.p99_bin < 256u ? s_val[q.p99_bin] : exp2(((double)q.p99_bin + 0.5) / (double)per_octave)) : 1.0;
  }
}

// ---- NEXT-2: L3 -------------------------------------------------------------------------------------------
// One CTA per key.  Shared memory: R (value, rank) pairs for the sort, the R scores.
__device__ __forceinline__ double normal_cdf(double z) { return 0.5 * erfc(-z * 0.7071067811865476); }

extern __shared__ unsigned char l3_smem[];

// bitonic sort of n (power of two) doubles with their payload, ascending; all threads of the CTA call
template <typename KT>
__device__ void bitonic_sort_simple(KT* v, uint16_t* id, uint32_t n) {
  for (uint32_t k = 2; k <= n; k <<= 1) {
    for (uint32_t j = k >> 1; j > 0; j >>= 1) {
      for (uint32_t i = threadIdx.x; i < n; i += blockDim.x) {
        const uint32_t p = i ^ j;
        if (p > i) {
          const bool up = (i & k) == 0u;
          const KT a = v[i], b = v[p];
          if ((a > b) == up && a != b) {
            v[i] = b; v[p] = a;
            const uint16_t t = id[i]; id[i] = id[p]; id[p] = t;
          }
        }
      }
      __syncthreads();
    }
  }
}

// The same network, four elements per thread: a thread that holds {i, i^jb, i^j, i^j^jb} (jb = j/2) runs the
// stages j and j/2 in registers, so two stages cost one trip through shared memory and one barrier (42 passes
// instead of 78 stages at n = 4096; every thread busy instead of half of them).  Identical compare-exchanges,
// hence identical output (ties included).  n >= 4, n / 4 <= blockDim.x.
template <typename KT>
__device__ void bitonic_sort(KT* v, uint16_t* id, uint32_t n) {
  if (n < 4u || (n >> 2) > blockDim.x) { bitonic_sort_simple(v, id, n); return; }
  const uint32_t t = threadIdx.x, nt = n >> 2;
  for (uint32_t k = 2; k <= n; k <<= 1) {
    uint32_t j = k >> 1;
    while (j >= 2u) {
      if (t < nt) {
        const uint32_t jb = j >> 1, b = (uint32_t)__ffs((int)jb) - 1u;
        const uint32_t base = ((t >> b) << (b + 2u)) | (t & (jb - 1u));
        const bool up = (base & k) == 0u;
        const uint32_t e[4] = {base, base | jb, base | j, base | j | jb};
        KT x[4];
        uint16_t q[4];
#pragma unroll
        for (int a = 0; a < 4; ++a) { x[a] = v[e[a]]; q[a] = id[e[a]]; }
#define ARGUS_CE(a, c)                                                         \
  if ((x[a] > x[c]) == up && x[a] != x[c]) {                                   \
    const KT tx = x[a]; x[a] = x[c]; x[c] = tx;                            \
    const uint16_t tq = q[a]; q[a] = q[c]; q[c] = tq;                          \
  }
        ARGUS_CE(0, 2) ARGUS_CE(1, 3) ARGUS_CE(0, 1) ARGUS_CE(2, 3)
#pragma unroll
        for (int a = 0; a < 4; ++a) { v[e[a]] = x[a]; id[e[a]] = q[a]; }
      }
      __syncthreads();
      j >>= 2;
    }
    if (j == 1u) {
      if (t < nt) {
        const uint32_t i = 4u * t;
        KT x[4];
        uint16_t q[4];
#pragma unroll
        for (int a = 0; a < 4; ++a) { x[a] = v[i + a]; q[a] = id[i + a]; }
        { const bool up = (i & k) == 0u; ARGUS_CE(0, 1) }
        { const bool up = ((i + 2u) & k) == 0u; ARGUS_CE(2, 3) }
#undef ARGUS_CE
#pragma unroll
        for (int a = 0; a < 4; ++a) { v[i + a] = x[a]; id[i + a] = q[a]; }
      }
      __syncthreads();
    }
  }
}

// Sum over b of |v_i - v_b| for every position i of the ascending array v[0..R) — the per-grid-point term of
// the mean-W1 score — from the GAPS g_i = v[i+1] - v[i] >= 0:  D_0 = sum_i g_i (R - 1 - i),
// D_{i+1} = D_i + g_i (2 i + 2 - R).  Every term is a gap times an integer, so ranks with identical CDF values
// get exactly equal sums (0 when all are equal); the prefix form F (2 i - R) + total - 2 pre[i] cancels instead.
// Block-wide: every thread owns PER consecutive positions; returns D of its positions in d[].
template <int PER>
__device__ __forceinline__ void abs_dev_sums(const double* v, uint32_t R, double* s_w, double* d) {
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5, nw = blockDim.x >> 5;
  const uint32_t i0 = threadIdx.x * PER;
  double h[PER], hsum = 0.0, d0 = 0.0;
#pragma unroll
  for (int k = 0; k < PER; ++k) {
    const uint32_t i = i0 + k;
    double g = 0.0;
    if (i + 1u < R) g = v[i + 1u] - v[i];
    h[k] = g * (double)((long long)(2u * i + 2u) - (long long)R);
    d0 += g * (double)(R - 1u - (i < R ? i : R - 1u));
    hsum += h[k];
  }
  // inclusive warp scans of hsum, warp totals of both
  double inc = hsum, tot0 = d0;
#pragma unroll
  for (int o = 1; o < 32; o <<= 1) {
    const double t = __shfl_up_sync(FULL, inc, o);
    if (lane >= o) inc += t;
  }
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) tot0 += __shfl_xor_sync(FULL, tot0, o);
  if (lane == 31) s_w[warp] = inc;
  if (lane == 0) s_w[32 + warp] = tot0;
  __syncthreads();
  double before = 0.0, D0 = 0.0;
  for (int w = 0; w < nw; ++w) {
    if (w < warp) before += s_w[w];
    D0 += s_w[32 + w];
  }
  double run = D0 + before + inc - hsum;          // D at this thread's first position
#pragma unroll
  for (int k = 0; k < PER; ++k) { d[k] = run; run += h[k]; }
  __syncthreads();                                 // s_w is reused by the next grid point
}

// One CTA of 1024 threads per key; R <= 4096: every thread owns at most 4 ranks (CDF evaluation) and at most 4
// sorted positions.  Per (rank, cluster) the log-normal parameters mu = ln p50, 1/sigma and the weight are
// computed once per key and kept in registers when the key has at most L3_CACHE (rank, cluster) pairs per thread
// (C = 1 at R = 4096, C <= 4 at R <= 1024), else recomputed per grid point.
constexpr int L3_CACHE = 4;
struct L3Par { double mu, isg, w; };               // isg = 1/sigma, 0 = a step at mu (R31)

__device__ __forceinline__ L3Par l3_par(uint32_t k, double tot, double p50, double p99) {
  L3Par q;
  q.mu = log(p50);
  const double sg = (log(p99) - q.mu) / 2.326;
  q.isg = sg > 0.0 ? 1.0 / sg : 0.0;
  q.w = (double)k / tot;
  return q;
}
// w Phi((lgx - mu) / sigma); |z| > 8.3: Phi differs from 0 / 1 by < 6e-17 (below half an ulp of the sums it enters)
__device__ __forceinline__ double l3_term(const L3Par& q, double lgx) {
  if (q.isg == 0.0) return lgx >= q.mu ? q.w : 0.0;
  const double z = (lgx - q.mu) * q.isg;
  if (z < -8.3) return 0.0;
  if (z > 8.3) return q.w;
  return q.w * normal_cdf(z);
}

// ---- ranks with identical mixtures ------------------------------------------------------------------------------
// The triples are quantised summaries (a bin stands for one duration, R30), so most ranks of a key carry the SAME
// mixture: same weights count_c / total, same p50, same p99 in every cluster slot, hence bit-identical CDF values
// at every grid point.  Grouping them first turns sum_b |F_a - F_b| over R ranks into a sum over the D distinct
// mixtures weighted by their multiplicities — exact algebra, no sort per grid point, O(D^2) instead of
// O(R log^2 R).  Classes are found by sorting a 64-bit hash of the mixture parameters and comparing neighbours
// field by field (a hash collision only splits work, it never merges two different mixtures).
constexpr uint32_t L3_MAX_CLASSES = 256;
constexpr uint32_t L3_CHUNK = 256;              // grid points per chunk of the class path
__device__ __forceinline__ unsigned long long l3_mix(unsigned long long h, unsigned long long v) {
  h ^= v; h *= 0x100000001b3ull; h ^= h >> 29;
  return h;
}
__device__ __forceinline__ double l3_total(const uint32_t* cnt, uint32_t r, uint32_t C) {
  double tot = 0.0;
  for (uint32_t c = 0; c < C; ++c) tot += (double)cnt[r * C + c];
  return tot;
}
__device__ unsigned long long l3_hash(const uint32_t* cnt, const double* p50, const double* p99, uint32_t r, uint32_t C) {
  const double tot = l3_total(cnt, r, C);
  unsigned long long h = 0xcbf29ce484222325ull;
  for (uint32_t c = 0; c < C; ++c) {
    const uint32_t k = cnt[r * C + c];
    if (k) {
      h = l3_mix(h, (unsigned long long)__double_as_longlong((double)k / tot));
      h = l3_mix(h, (unsigned long long)__double_as_longlong(p50[r * C + c]));
      h = l3_mix(h, (unsigned long long)__double_as_longlong(p99[r * C + c]));
    } else {
      h = l3_mix(h, 0x9e3779b97f4a7c15ull);
    }
  }
  return h & 0x7FFFFFFFFFFFFFFFull;            // the padding key (all ones) sorts behind every rank
}
__device__ bool l3_same_mixture(const uint32_t* cnt, const double* p50, const double* p99, uint32_t a, uint32_t b, uint32_t C) {
  const double ta = l3_total(cnt, a, C), tb = l3_total(cnt, b, C);
  for (uint32_t c = 0; c < C; ++c) {
    const uint32_t ka = cnt[a * C + c], kb = cnt[b * C + c];
    if ((ka == 0u) != (kb == 0u)) return false;
    if (ka == 0u) continue;
    if (__double_as_longlong((double)ka / ta) != __double_as_longlong((double)kb / tb)) return false;
    if (__double_as_longlong(p50[a * C + c]) != __double_as_longlong(p50[b * C + c])) return false;
    if (__double_as_longlong(p99[a * C + c]) != __double_as_longlong(p99[b * C + c])) return false;
  }
  return true;
}
// F_r(x) of eq. (2) for one rank, parameters recomputed (the class path evaluates a handful of ranks only)
__device__ double l3_cdf_of(const uint32_t* cnt, const double* p50, const double* p99, uint32_t r, uint32_t C, double lgx) {
  const double tot = l3_total(cnt, r, C);
  double F = 0.0;
  if (tot > 0.0)
    for (uint32_t c = 0; c < C; ++c) {
      const uint32_t k = cnt[r * C + c];
      if (k) F += l3_term(l3_par(k, tot, p50[r * C + c], p99[r * C + c]), lgx);
    }
  return F;
}

__global__ void __launch_bounds__(1024)
l3_kernel(argus_l3_in in, argus_l3_params P, double* __restrict__ score_out, argus_l3_stat* __restrict__ stat_out,
          uint8_t* __restrict__ flags_out, unsigned long long* __restrict__ path_count) {
  const uint32_t R = in.n_ranks, C = in.max_clusters, key = blockIdx.x, G = P.n_grid;
  uint32_t n2 = 1;
  while (n2 < R) n2 <<= 1;
  double* val = reinterpret_cast<double*>(l3_smem);                 // [n2]
  double* score = val + n2;                                         // [R]
  uint16_t* id = reinterpret_cast<uint16_t*>(score + R);            // [n2]
  uint16_t* class_of = id + n2;                                     // [n2]: class of every rank (class path)
  __shared__ double s_red[64];
  __shared__ uint16_t s_rep[L3_MAX_CLASSES];                         // a rank of every class
  __shared__ uint32_t s_mult[L3_MAX_CLASSES];                        // ranks in every class
  __shared__ double s_sc[L3_MAX_CLASSES];
  __shared__ double s_wj[L3_CHUNK], s_lg[L3_CHUNK];                  // trapezoid weight and log x of a chunk of grid points
  __shared__ double s_part[1024];
  __shared__ uint32_t s_scan[33];
  __shared__ double s_lo, s_hi, s_fence;
  const uint32_t* cnt = in.count + (size_t)key * R * C;
  const double* p50 = in.p50 + (size_t)key * R * C;
  const double* p99 = in.p99 + (size_t)key * R * C;
  // grid bounds (R32): 0.5 * min p50 .. 2 * max p99 over the clusters with count > 0
  double mn = INFINITY, mx = 0.0;
  for (uint32_t i = threadIdx.x; i < R * C; i += blockDim.x)
    if (cnt[i]) { mn = fmin(mn, p50[i]); mx = fmax(mx, p99[i]); }
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) { mn = fmin(mn, __shfl_xor_sync(FULL, mn, o)); mx = fmax(mx, __shfl_xor_sync(FULL, mx, o)); }
  if ((threadIdx.x & 31) == 0) { s_red[threadIdx.x >> 5] = mn; s_red[32 + (threadIdx.x >> 5)] = mx; }
  for (uint32_t r = threadIdx.x; r < R; r += blockDim.x) score[r] = 0.0;
  __syncthreads();
  if (threadIdx.x == 0) {
    double a = INFINITY, b = 0.0;
    for (uint32_t w = 0; w < (blockDim.x + 31u) / 32u; ++w) { a = fmin(a, s_red[w]); b = fmax(b, s_red[32 + w]); }
    s_lo = a; s_hi = b;
  }
  __syncthreads();
  const bool empty = !(s_hi > 0.0);
  bool by_class = false;
  if (!empty) {
    // ---- classes of identical mixtures ------------------------------------------------------------------
    unsigned long long* hkey = reinterpret_cast<unsigned long long*>(val);
    for (uint32_t r = threadIdx.x; r < n2; r += blockDim.x) {
      hkey[r] = r < R ? l3_hash(cnt, p50, p99, r, C) : ~0ull;
      id[r] = (uint16_t)r;
    }
    for (uint32_t d = threadIdx.x; d < L3_MAX_CLASSES; d += blockDim.x) { s_mult[d] = 0u; s_sc[d] = 0.0; }
    __syncthreads();
    bitonic_sort(hkey, id, n2);
    // sorted position i opens a class unless its mixture equals its left neighbour's; PER consecutive positions
    // per thread, block-wide inclusive scan of the flags
    const uint32_t PER = (n2 + blockDim.x - 1u) / blockDim.x;
    uint32_t fl[4] = {0u, 0u, 0u, 0u}, loc = 0u;
    for (uint32_t k = 0; k < PER; ++k) {
      const uint32_t i = threadIdx.x * PER + k;
      if (i < R) {
        fl[k] = (i == 0u || hkey[i] != hkey[i - 1u] || !l3_same_mixture(cnt, p50, p99, id[i], id[i - 1u], C)) ? 1u : 0u;
        loc += fl[k];
      }
    }
    uint32_t inc = loc;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
      const uint32_t v = __shfl_up_sync(FULL, inc, o);
      if ((threadIdx.x & 31) >= (uint32_t)o) inc += v;
    }
    if ((threadIdx.x & 31) == 31) s_scan[threadIdx.x >> 5] = inc;
    __syncthreads();
    uint32_t before = 0u, n_cls = 0u;
    for (uint32_t w = 0; w < (blockDim.x >> 5); ++w) {
      if (w < (threadIdx.x >> 5)) before += s_scan[w];
      n_cls += s_scan[w];
    }
    by_class = n_cls <= L3_MAX_CLASSES;
    if (by_class) {
      uint32_t run = before + inc - loc;                   // classes opened before this thread's first position
      for (uint32_t k = 0; k < PER; ++k) {
        const uint32_t i = threadIdx.x * PER + k;
        if (i < R) {
          run += fl[k];
          const uint32_t c = run - 1u;
          class_of[id[i]] = (uint16_t)c;
          if (fl[k]) s_rep[c] = id[i];
          atomicAdd(&s_mult[c], 1u);
        }
      }
      __syncthreads();
      // Grid points in chunks of JB: (1) the chunk's abscissae and trapezoid weights, one thread each; (2) eq. 2 for
      // every (class, grid point) pair of the chunk, all threads; (3) thread (class d, group g) sums
      // w_j sum_b m_b |F_d - F_b| over the grid points j = g, g + groups, ...; (4) thread d adds its groups'
      // partial sums in a fixed order.  No atomics: the result does not depend on scheduling.
      const double llo = log(0.5 * s_lo), lhi = log(2.0 * s_hi);
      uint32_t JB = n2 / n_cls;
      JB = JB > L3_CHUNK ? L3_CHUNK : JB;
      const uint32_t groups = blockDim.x / n_cls;                  // >= 1: n_cls <= min(R, 256) <= blockDim.x
      const uint32_t my_d = threadIdx.x % n_cls, my_g = threadIdx.x / n_cls;
      for (uint32_t j0 = 0; j0 < G; j0 += JB) {
        const uint32_t nj = G - j0 < JB ? G - j0 : JB;
        for (uint32_t jj = threadIdx.x; jj < nj; jj += blockDim.x) {
          const uint32_t j = j0 + jj;
          const double lx = llo + (lhi - llo) * (double)j / (double)(G - 1u);
          const double x = exp(lx);
          const double xm = j ? exp(llo + (lhi - llo) * (double)(j - 1u) / (double)(G - 1u)) : x;
          const double xp = j + 1u < G ? exp(llo + (lhi - llo) * (double)(j + 1u) / (double)(G - 1u)) : x;
          s_wj[jj] = 0.5 * (xp - xm);
          s_lg[jj] = log(x);                               // log(x) of the oracle is log(exp(lx)): take it the same way
        }
        __syncthreads();
        for (uint32_t p = threadIdx.x; p < n_cls * nj; p += blockDim.x) {
          const uint32_t d = p % n_cls, jj = p / n_cls;
          val[p] = l3_cdf_of(cnt, p50, p99, s_rep[d], C, s_lg[jj]);      // val[jj * n_cls + d]
        }
        __syncthreads();
        double acc = 0.0;
        if (my_g < groups)
          for (uint32_t jj = my_g; jj < nj; jj += groups) {
            const double* row = val + (size_t)jj * n_cls;
            const double fd = row[my_d];
            double s = 0.0;
            for (uint32_t b2 = 0; b2 < n_cls; ++b2) s += (double)s_mult[b2] * fabs(fd - row[b2]);
            acc += s_wj[jj] * s;
          }
        s_part[threadIdx.x] = acc;
        __syncthreads();
        if (threadIdx.x < n_cls) {
          double s = s_sc[threadIdx.x];
          for (uint32_t g2 = 0; g2 < groups; ++g2) s += s_part[g2 * n_cls + threadIdx.x];
          s_sc[threadIdx.x] = s;
        }
        __syncthreads();
      }
      for (uint32_t r = threadIdx.x; r < R; r += blockDim.x) score[r] = s_sc[class_of[r]];
    }
    __syncthreads();
  }
  // which way this key went (argus_l3_path_count): [0] ranks fell into <= 256 classes of identical mixtures,
  // [1] the general path below (a sort of R CDF values per grid point), [2] no cluster at all
  if (threadIdx.x == 0 && path_count) atomicAdd(&path_count[empty ? 2 : (by_class ? 0 : 1)], 1ull);
  if (!empty && !by_class) {
    // per-thread totals and, when they fit, the cached parameters of this thread's NON-EMPTY (rank, cluster)
    // pairs in (rank slot, cluster) order — the order the sums below take; a thread with more than L3_CACHE of
    // them recomputes its parameters at every grid point
    L3Par par[L3_CACHE];
    uint32_t slot[L3_CACHE];
    uint32_t n_ent = 0;
    double tot[4] = {0.0, 0.0, 0.0, 0.0};
#pragma unroll
    for (int a = 0; a < 4; ++a) {
      const uint32_t r = threadIdx.x + (uint32_t)a * blockDim.x;
      if (r < R)
        for (uint32_t c = 0; c < C; ++c) tot[a] += (double)cnt[r * C + c];
    }
#pragma unroll
    for (int q = 0; q < L3_CACHE; ++q) { par[q].mu = 0.0; par[q].isg = 0.0; par[q].w = 0.0; slot[q] = 4u; }
#pragma unroll
    for (int a = 0; a < 4; ++a) {
      const uint32_t r = threadIdx.x + (uint32_t)a * blockDim.x;
      if (r < R && tot[a] > 0.0)
        for (uint32_t c = 0; c < C; ++c) {
          const uint32_t k = cnt[r * C + c];
          if (k) {
            if (n_ent < (uint32_t)L3_CACHE) {
              const L3Par v = l3_par(k, tot[a], p50[r * C + c], p99[r * C + c]);
#pragma unroll
              for (int q = 0; q < L3_CACHE; ++q)
                if ((uint32_t)q == n_ent) { par[q] = v; slot[q] = (uint32_t)a; }
            }
            ++n_ent;
          }
        }
    }
    const bool cached = n_ent <= (uint32_t)L3_CACHE;
    const double llo = log(0.5 * s_lo), lhi = log(2.0 * s_hi);
    for (uint32_t j = 0; j < G; ++j) {
      const double lx = llo + (lhi - llo) * (double)j / (double)(G - 1u);
      const double x = exp(lx);
      // trapezoid weight of grid point j: half the two neighbouring intervals (eq. 3 on a log-uniform grid)
      const double xm = j ? exp(llo + (lhi - llo) * (double)(j - 1u) / (double)(G - 1u)) : x;
      const double xp = j + 1u < G ? exp(llo + (lhi - llo) * (double)(j + 1u) / (double)(G - 1u)) : x;
      const double wj = 0.5 * (xp - xm);
      // F_r(x_j), eq. (2); log(x) of the oracle is log(exp(lx)): take it the same way
      const double lgx = log(x);
      double Fa[4] = {0.0, 0.0, 0.0, 0.0};
      if (cached) {
#pragma unroll
        for (int q = 0; q < L3_CACHE; ++q) {
          if (slot[q] < 4u) {
            const double tq = l3_term(par[q], lgx);
#pragma unroll
            for (int a = 0; a < 4; ++a) if (slot[q] == (uint32_t)a) Fa[a] += tq;
          }
        }
      } else {
#pragma unroll
        for (int a = 0; a < 4; ++a) {
          const uint32_t r = threadIdx.x + (uint32_t)a * blockDim.x;
          if (r < R && tot[a] > 0.0)
            for (uint32_t c = 0; c < C; ++c) {
              const uint32_t k = cnt[r * C + c];
              if (k) Fa[a] += l3_term(l3_par(k, tot[a], p50[r * C + c], p99[r * C + c]), lgx);
            }
        }
      }
      bool same = true;                            // every value of this thread equals rank 0's?
#pragma unroll
      for (int a = 0; a < 4; ++a) {
        const uint32_t r = threadIdx.x + (uint32_t)a * blockDim.x;
        if (r < n2) {
          val[r] = r < R ? Fa[a] : INFINITY;       // padding sorts to the end
          id[r] = (uint16_t)r;
        }
      }
      __syncthreads();
      {
        const double f0 = val[0];
#pragma unroll
        for (int a = 0; a < 4; ++a) {
          const uint32_t r = threadIdx.x + (uint32_t)a * blockDim.x;
          if (r < R) same = same && Fa[a] == f0;
        }
      }
      // all ranks agree at this grid point (below every distribution, above every one, or identical triples):
      // every |F_a - F_b| is 0, nothing to sort and nothing to add
      if (__syncthreads_and(same)) continue;
      bitonic_sort(val, id, n2);
      // sum_b |F_r - F_b| at every sorted position, from the gaps
      double d[4];
      if (n2 >= 4096u) {
        abs_dev_sums<4>(val, R, s_red, d);
        for (int k = 0; k < 4; ++k) { const uint32_t i = threadIdx.x * 4u + k; if (i < R) score[id[i]] += wj * d[k]; }
      } else if (n2 >= 2048u) {
        abs_dev_sums<2>(val, R, s_red, d);
        for (int k = 0; k < 2; ++k) { const uint32_t i = threadIdx.x * 2u + k; if (i < R) score[id[i]] += wj * d[k]; }
      } else {
        abs_dev_sums<1>(val, R, s_red, d);
        if (threadIdx.x < R) score[id[threadIdx.x]] += wj * d[0];
      }
      __syncthreads();
    }
  }
  // deviation score = mean W1 to the other ranks; quartiles by linear interpolation (R33)
  const double inv = R > 1u ? 1.0 / (double)(R - 1u) : 1.0;
  for (uint32_t r = threadIdx.x; r < n2; r += blockDim.x) {
    if (r < R) {
      score[r] *= inv;
      score_out[(size_t)key * R + r] = score[r];
      val[r] = score[r];
    } else {
      val[r] = INFINITY;
    }
    id[r] = (uint16_t)r;
  }
  __syncthreads();
  bitonic_sort(val, id, n2);
  if (threadIdx.x == 0) {
    auto quant = [&](double q) {
      const double pos = q * (double)(R - 1u);
      const uint32_t i0 = (uint32_t)floor(pos);
      const double fr = pos - (double)i0;
      const uint32_t i1 = i0 + 1u < R ? i0 + 1u : i0;
      return val[i0] + fr * (val[i1] - val[i0]);
    };
    const double q1 = quant(0.25), q3 = quant(0.75);
    s_fence = q3 + P.alpha * (q3 - q1);                              // eq. (4)
    argus_l3_stat st;
    st.q1 = q1; st.q3 = q3; st.fence = s_fence;
    st.x_lo = empty ? 1.0 : 0.5 * s_lo; st.x_hi = empty ? 1.0 : 2.0 * s_hi;
    stat_out[key] = st;
  }
  __syncthreads();
  const double fence = s_fence;
  for (uint32_t r = threadIdx.x; r < R; r += blockDim.x) flags_out[(size_t)key * R + r] = score[r] > fence ? 1 : 0;
}

// ---- NEXT-3: L2 ---------------------------------------------------------------------------------------------
// One CTA per routed event k (phase span, index P = whole iteration): x_r = mean over the T steps of span_ns.
// Group sums are taken in a FIXED order (no floating-point atomics): the member count of every group comes from
// integer atomics, a group of one is its member's value, and every larger group is summed by one warp — lane l
// adds its members r = l, l + 32, ... in ascending order, then the 32 partial sums meet in a fixed shuffle tree —
// so that mu, sigma, CV, z and with them the CV class and the z > threshold flag are the same bits in every run.
__device__ __forceinline__ double l2_group_sum(const uint32_t* __restrict__ gid, const double* xb, uint32_t first, uint32_t last,
                                               uint32_t g, double mu, bool squared) {
  const uint32_t lane = threadIdx.x & 31u;
  double acc = 0.0;
  for (uint32_t r = first + lane; r <= last; r += 32u)      // only the span of ranks that holds the group's members
    if (gid[r] == g) {
      const double d = squared ? xb[r] - mu : xb[r];
      acc += squared ? d * d : d;
    }
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) acc += __shfl_xor_sync(0xFFFFFFFFu, acc, o);   // xor tree: all lanes, same order
  return acc;
}

__global__ void __launch_bounds__(1024)
l2_kernel(const uint8_t* __restrict__ records, argus_dims D, const uint8_t* __restrict__ route, uint32_t n_dims,
          const uint32_t* __restrict__ group_id, double z_thr, argus_l2_group* __restrict__ groups,
          double* __restrict__ z_out, uint8_t* __restrict__ flag_out, double* __restrict__ xbar_ws) {
  const uint32_t k = blockIdx.x, R = D.R;
  const bool routed = route[k] < n_dims;          // a route byte beyond the dimensions given: the event joins no group
  const uint32_t* gid = group_id + (size_t)(routed ? route[k] : 0u) * R;
  argus_l2_group* G = groups + (size_t)k * R;
  double* xb = xbar_ws + (size_t)k * R;
  for (uint32_t r = threadIdx.x; r < R; r += blockDim.x) {
    double s = 0.0;
    for (uint32_t t = 0; t < D.T; ++t) {
      const argus_span* sp = reinterpret_cast<const argus_span*>(records + ((size_t)r * D.T + t) * D.rec_bytes + D.span_off) + k;
      s += (double)sp->span_ns;
    }
    xb[r] = s / (double)D.T;
    argus_l2_group g;
    g.n = 0u; g.cls = 0xFFFFFFFFu; g.mu = 0.0; g.sigma = 0.0; g.cv = 0.0;
    G[r] = g;
  }
  __threadfence();
  __syncthreads();
  // member count, first and last member of every group: integer atomics, exact whatever the order.  Until the
  // group's entry is written below, its cls word holds the first member and the low word of cv the last one.
  for (uint32_t r = threadIdx.x; r < R; r += blockDim.x)
    if (routed && gid[r] < R) {
      argus_l2_group* q = &G[gid[r]];
      atomicAdd(&q->n, 1u);
      atomicMin(&q->cls, r);
      atomicMax(reinterpret_cast<uint32_t*>(&q->cv), r);
    }
  __threadfence();
  __syncthreads();
  const uint32_t warp = threadIdx.x >> 5, n_warps = blockDim.x >> 5, lane = threadIdx.x & 31u;
  for (uint32_t g = warp; g < R; g += n_warps) {
    const uint32_t n = G[g].n;
    if (n == 0u) {                                          // no such group: the entry reads n = 0 and zeros
      if (lane == 0u) G[g].cls = 0u;
      continue;
    }
    const uint32_t first = G[g].cls, last = *reinterpret_cast<const uint32_t*>(&G[g].cv);
    __syncwarp();                                           // every lane has read the bounds before lane 0 overwrites them
    argus_l2_group q;
    q.n = n;
    q.mu = l2_group_sum(gid, xb, first, last, g, 0.0, false) / (double)n;
    const double ss = n > 1u ? l2_group_sum(gid, xb, first, last, g, q.mu, true) : 0.0;
    q.sigma = n > 1u ? sqrt(ss / (double)(n - 1u)) : 0.0;                       // eq. (5): |G| - 1
    q.cv = (q.mu > 0.0 && q.sigma > 0.0) ? q.sigma / q.mu : 0.0;                // R34
    q.cls = q.cv < 0.02 ? 0u : (q.cv < 0.05 ? 1u : 2u);
    if (lane == 0u) G[g] = q;
  }
  __threadfence();
  __syncthreads();
  for (uint32_t r = threadIdx.x; r < R; r += blockDim.x) {
    double z = 0.0;
    if (routed && gid[r] < R) {
      const argus_l2_group q = G[gid[r]];
      if (q.sigma > 0.0) z = (xb[r] - q.mu) / q.sigma;
    }
    z_out[(size_t)k * R + r] = z;
    flag_out[(size_t)k * R + r] = z > z_thr ? 1 : 0;
  }
}

// ---- NEXT-3: L1, one warp per series -----------------------------------------------------------------------
__device__ __forceinline__ double series_at(const uint8_t* base, uint64_t sstride, uint64_t tstride, uint32_t s, uint32_t t) {
  return (double)*reinterpret_cast<const unsigned long long*>(base + (size_t)s * sstride + (size_t)t * tstride);
}

// median (mean of the two middle values for an even count) of the points of x outside [a, b], by rank counting
__device__ double median_outside(const double* x, uint32_t T, uint32_t a, uint32_t b) {
  const int lane = threadIdx.x & 31;
  const uint32_t n = T - (b - a + 1u);
  if (n == 0u) return 0.0;
  const uint32_t k_hi = n / 2u, k_lo = (n & 1u) ? k_hi : k_hi - 1u;
  double v_lo = 0.0, v_hi = 0.0;
  for (uint32_t i = lane; i < ((T + 31u) & ~31u); i += 32) {
    bool f_lo = false, f_hi = false;
    double v = 0.0;
    if (i < T && (i < a || i > b)) {
      v = x[i];
      uint32_t less = 0, eq = 0;
      for (uint32_t q = 0; q < T; ++q)
        if (q < a || q > b) { less += x[q] < v; eq += x[q] == v; }
      f_lo = less <= k_lo && k_lo < less + eq;
      f_hi = less <= k_hi && k_hi < less + eq;
    }
    const uint32_t m_lo = __ballot_sync(FULL, f_lo), m_hi = __ballot_sync(FULL, f_hi);
    if (m_lo) v_lo = __shfl_sync(FULL, v, __ffs((int)m_lo) - 1);
    if (m_hi) v_hi = __shfl_sync(FULL, v, __ffs((int)m_hi) - 1);
  }
  return (n & 1u) ? v_hi : 0.5 * (v_lo + v_hi);
}

extern __shared__ double l1_smem[];

__global__ void __launch_bounds__(128)
l1_kernel(const uint8_t* __restrict__ base, uint64_t sstride, uint64_t tstride, uint32_t n_series, uint32_t T,
          argus_l1_params P, argus_l1_out* __restrict__ out) {
  const int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
  const uint32_t s = blockIdx.x * 4u + (uint32_t)w;
  if (s >= n_series) return;
  double* x = l1_smem + (size_t)w * (2u * T);               // T values, then T candidate marks (as doubles: 0 / 1)
  double* mark = x + T;
  for (uint32_t t = lane; t < T; t += 32) { x[t] = series_at(base, sstride, tstride, s, t); mark[t] = 0.0; }
  __syncwarp();
  argus_l1_out o;
  memset(&o, 0, sizeof o);
  // ---- jitter, phase 1: windows whose max/min exceeds theta mark their points
  const uint32_t W = P.window;
  if (T >= W) {
    for (uint32_t i = lane; i + W <= T; i += 32) {
      double mn = x[i], mx = x[i];
      for (uint32_t q = 1; q < W; ++q) { mn = fmin(mn, x[i + q]); mx = fmax(mx, x[i + q]); }
      if (mx > P.theta * mn)
        for (uint32_t q = 0; q < W; ++q) mark[i + q] = 1.0;      // benign race: everybody writes 1
    }
  }
  __syncwarp();
  // adjacent or overlapping candidate windows merge = maximal runs of marked points; phase 2 per run
  uint32_t n_int = 0, t0 = 0;
  bool any_width = false;
  while (t0 < T) {
    if (mark[t0] == 0.0) { ++t0; continue; }
    uint32_t t1 = t0;
    while (t1 + 1u < T && mark[t1 + 1u] != 0.0) ++t1;
    const double basel = median_outside(x, T, t0, t1);
    uint32_t best = 0, run = 0;
    for (uint32_t t = t0; t <= t1; ++t) {            // every lane walks the run (it is short): uniform result
      run = x[t] > P.beta * basel ? run + 1u : 0u;
      best = run > best ? run : best;
    }
    if (n_int < ARGUS_L1_MAX_INTERVALS) {
      o.interval[n_int].first = t0; o.interval[n_int].last = t1; o.interval[n_int].width = best;
      o.interval[n_int].baseline = basel;
    }
    ++n_int;
    any_width |= best > 0u;
    t0 = t1 + 1u;
  }
  o.n_intervals = n_int;
  // ---- change point: lanes share the splits, two passes per side as the oracle
  double best_ratio = 0.0;
  uint32_t best_t = 0;
  const uint32_t m = P.min_seg;
  if (T >= 2u * m) {
    for (uint32_t t = m + lane; t + m <= T; t += 32) {
      double sL = 0.0, sR = 0.0;
      for (uint32_t q = 0; q < t; ++q) sL += x[q];
      for (uint32_t q = t; q < T; ++q) sR += x[q];
      const double muL = sL / (double)t, muR = sR / (double)(T - t);
      if (!(muL > 0.0) || !(muR > 0.0)) continue;
      double vL = 0.0, vR = 0.0;
      for (uint32_t q = 0; q < t; ++q) vL += (x[q] - muL) * (x[q] - muL);
      for (uint32_t q = t; q < T; ++q) vR += (x[q] - muR) * (x[q] - muR);
      const double sdL = sqrt(vL / (double)(t - 1u)), sdR = sqrt(vR / (double)(T - t - 1u));
      const double ratio = muR / muL;
      if (ratio > P.ratio_min && sdL / muL < P.rsd_max && sdR / muR < P.rsd_max && ratio > best_ratio) {
        best_ratio = ratio; best_t = t;
      }
    }
  }
  // the largest ratio wins, the earliest split among equals
#pragma unroll
  for (int ofs = 16; ofs > 0; ofs >>= 1) {
    const double r2 = __shfl_xor_sync(FULL, best_ratio, ofs);
    const uint32_t t2 = __shfl_xor_sync(FULL, best_t, ofs);
    if (r2 > best_ratio || (r2 == best_ratio && r2 > 0.0 && t2 < best_t)) { best_ratio = r2; best_t = t2; }
  }
  o.cp_found = best_ratio > 0.0 ? 1u : 0u;
  o.cp_step = best_t;
  o.cp_ratio = best_ratio;
  o.cls = (any_width ? 1u : 0u) | (o.cp_found ? 2u : 0u);     // stable / jitter / regression / both
  if (lane == 0) out[s] = o;
}

}  // namespace

// ---- launchers ---------------------------------------------------------------------------------------------
cudaError_t argus_launch_fine_hist(argus_ctx* ctx, const argus_event* ev, uint64_t n, uint32_t* d_hist, cudaStream_t s) {
  if (n == 0) return cudaSuccess;
  uint64_t blocks = (n + 255) / 256;
  const uint64_t cap = (uint64_t)ctx->sm_count * 16;
  if (blocks > cap) blocks = cap;
  fine_hist_kernel<<<(unsigned)blocks, 256, 0, s>>>(reinterpret_cast<const uint4*>(ev), n, ctx->dims, d_hist);
  ctx->n_kernels += 1;
  return cudaGetLastError();
}

cudaError_t argus_launch_kde_hist(argus_ctx* ctx, const uint32_t* d_hist, uint64_t n_cells, const argus_kde_params* P,
                                  argus_cluster* d_clusters, uint8_t* d_n, double* d_density, cudaStream_t s) {
  if (n_cells == 0) return cudaSuccess;
  kde_hist_kernel<<<(unsigned)((n_cells + 31) / 32), 256, 0, s>>>(d_hist, n_cells, *P, d_clusters, d_n, d_density);
  ctx->n_kernels += 1;
  return cudaGetLastError();
}

cudaError_t argus_launch_kde_records(argus_ctx* ctx, const void* d_records, const argus_kde_params* P,
                                     argus_cluster* d_clusters, uint8_t* d_n, cudaStream_t s) {
  const uint64_t n_cells = (uint64_t)ctx->dims.R * ctx->dims.T * ctx->dims.S;
  kde_records_kernel<<<(unsigned)((n_cells + KDE_REC_NT - 1) / KDE_REC_NT), KDE_REC_NT, 0, s>>>(
      static_cast<const uint8_t*>(d_records), ctx->dims, *P, d_clusters, d_n);
  ctx->n_kernels += 1;
  return cudaGetLastError();
}

cudaError_t argus_launch_clusters_to_l3(argus_ctx* ctx, const argus_cluster* d_clusters, uint32_t mc, uint32_t per_octave,
                                        uint32_t* d_count, double* d_p50, double* d_p99, cudaStream_t s) {
  clusters_to_l3_kernel<<<(unsigned)ctx->sm_count * 8u, 256, 0, s>>>(d_clusters, ctx->dims, mc, per_octave, d_count, d_p50,
                                                                    d_p99);
  ctx->n_kernels += 1;
  return cudaGetLastError();
}

size_t argus_l3_smem_bytes(uint32_t R) {
  uint32_t n2 = 1;
  while (n2 < R) n2 <<= 1;
  return sizeof(double) * ((size_t)n2 + R) + sizeof(uint16_t) * 2u * n2;
}

cudaError_t argus_configure_paper_literal(argus_ctx* ctx) {
  cudaError_t e = argus_optin_all_smem(l3_kernel, ctx->max_smem_optin);
  return e == cudaSuccess ? argus_optin_all_smem(l1_kernel, ctx->max_smem_optin) : e;
}

cudaError_t argus_launch_l3(argus_ctx* ctx, const argus_l3_in* in, const argus_l3_params* P, double* d_score,
                            argus_l3_stat* d_stat, uint8_t* d_flags, cudaStream_t s) {
  if (in->n_keys == 0) return cudaSuccess;
  const size_t smem = argus_l3_smem_bytes(in->n_ranks);
  // one CTA per key: every thread owns <= 4 ranks, and a rank each in the scan when R <= 1024 — small jobs get
  // small CTAs, so that several keys share an SM
  uint32_t n2 = 1;
  while (n2 < in->n_ranks) n2 <<= 1;
  const unsigned threads = n2 >= 1024u ? 1024u : (n2 < 64u ? 64u : n2);
  l3_kernel<<<in->n_keys, threads, smem, s>>>(*in, *P, d_score, d_stat, d_flags, ctx->d_counters + 4);
  ctx->n_kernels += 1;
  return cudaGetLastError();
}

cudaError_t argus_launch_l2(argus_ctx* ctx, const void* d_records, const uint8_t* d_route, uint32_t n_dims,
                            const uint32_t* d_group_id, double z_thr, argus_l2_group* d_groups, double* d_z, uint8_t* d_flags, double* d_xbar,
                            cudaStream_t s) {
  // few CTAs (one per routed event), each a chain of strided loads and fenced phases: as many threads as a CTA takes
  l2_kernel<<<ctx->dims.P + 1u, ctx->dims.R >= 1024u ? 1024 : 256, 0, s>>>(static_cast<const uint8_t*>(d_records), ctx->dims, d_route, n_dims, d_group_id, z_thr,
                                             d_groups, d_z, d_flags, d_xbar);
  ctx->n_kernels += 1;
  return cudaGetLastError();
}

cudaError_t argus_launch_l1(argus_ctx* ctx, const void* d_base, uint64_t sstride, uint64_t tstride, uint32_t n_series,
                            uint32_t T, const argus_l1_params* P, argus_l1_out* d_out, cudaStream_t s) {
  if (n_series == 0 || T == 0) return cudaSuccess;
  const size_t smem = sizeof(double) * 2u * T * 4u;
  l1_kernel<<<(n_series + 3u) / 4u, 128, smem, s>>>(static_cast<const uint8_t*>(d_base), sstride, tstride, n_series, T, *P,
                                                   d_out);
  ctx->n_kernels += 1;
  return cudaGetLastError();
}
