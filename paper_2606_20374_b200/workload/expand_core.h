/* expand_core.h — the seeded synthetic-workload expander (input generator).
 *
 * This module serves both the CPU oracle tests and the CUDA path with the SAME event bytes and
 * holds none of the method's arithmetic (no bucketing, no summaries, no medians).  It is integer
 * only, so the host build (gcc) and the device build (nvcc) of this one source produce identical
 * bytes; all floating point lives in recipe.py, which builds the lookup tables once per run.
 *
 * Shape (stands in for the paper's production traces, which are not public): each stream of a
 * rank replays a fixed kernel sequence shared by all ranks, same-position
 * durations are consistent up to a small log-normal jitter, streams are serial
 * timelines merged by start time, phases are consecutive runs of a step.
 */
#ifndef WL_EXPAND_CORE_H_
#define WL_EXPAND_CORE_H_
#include <stdint.h>

#ifdef __CUDACC__
#define WL_HD __host__ __device__ __forceinline__
#else
#define WL_HD static inline
#endif

#define WL_MAX_STREAMS 16
#define WL_JIT_BITS 12   /* jitter / gap quantile tables: 4096 entries */
#define WL_PAR_BITS 16   /* pareto ratio table: 65536 entries          */

typedef struct wl_event {      /* the 32-byte record of NS */
  uint32_t rank, step, sig;
  uint16_t stream, phase;
  int64_t  start_ns, end_ns;
} wl_event;

typedef struct wl_fault {      /* dur *= mult_q16 / 65536 when every selector matches */
  uint32_t rank;
  uint32_t step;       /* 0xFFFFFFFF = all steps (relative step index t) */
  uint32_t sig;        /* 0xFFFFFFFF = any sig   */
  uint32_t sig_class;  /* 0xFFFFFFFF = any class; else wl_sig_class(sig) */
  uint32_t phase;      /* 0xFFFFFFFF = any phase */
  uint32_t mult_q16;
} wl_fault;

typedef struct wl_desc {
  uint64_t seed;
  uint32_t n_ranks, n_steps, n_events, n_sigs, n_phases, n_streams; /* R, T, N, S, P, streams */
  uint32_t step_base;
  uint32_t dur_mode;      /* 0: base[sig]*jitter   1: pareto per event (xmin_ns, pareto_q16) */
  uint32_t shuffle;       /* 1: scatter every event to wl_perm(global index) (config 3) */
  uint32_t n_faults;
  uint64_t xmin_ns;
  uint64_t step_gap_ns;   /* idle time between a rank's consecutive steps */
  /* tables (host pointers for the host expander, device pointers for the device one) */
  const uint32_t* prog_sig;    /* [T][N]  per step: streams' sequences concatenated            */
  const uint32_t* prog_off;    /* [T][n_streams+1] offsets of each stream's sequence in prog_sig */
  const uint16_t* stream_id;   /* [n_streams] id written into the record                        */
  const uint64_t* base_ns;     /* [S]                                                            */
  const uint32_t* jit_q16;     /* [4096] jitter multiplier quantiles, Q16                        */
  const uint32_t* gap_ns;      /* [4096] inter-kernel gap quantiles                              */
  const uint32_t* pareto_q16;  /* [65536] Pareto(alpha) ratio quantiles, Q16 (dur_mode 1)        */
  const wl_fault* faults;      /* [n_faults] sorted by rank                                      */
  const uint32_t* fault_off;   /* [R+1] faults of rank r are faults[fault_off[r]..fault_off[r+1]) */
  const uint32_t* mode2_q16;   /* [S] 0 = unimodal sig; else the multiplier (Q16) of the sig's SECOND duration
                                  mode, taken by half of its events (same-name kernels "differ in
                                  duration by several multiples" across positions) */
} wl_desc;

WL_HD uint64_t wl_mix(uint64_t x) {            /* splitmix64 finaliser */
  x ^= x >> 30; x *= 0xBF58476D1CE4E5B9ull;
  x ^= x >> 27; x *= 0x94D049BB133111EBull;
  x ^= x >> 31; return x;
}
WL_HD uint64_t wl_hash(uint64_t seed, uint32_t rank, uint32_t t, uint32_t j, uint32_t i) {
  uint64_t h = wl_mix(seed + 0x9E3779B97F4A7C15ull * (uint64_t)(rank + 1));
  h = wl_mix(h ^ (((uint64_t)t << 32) | (uint64_t)j));
  return wl_mix(h + 0x9E3779B97F4A7C15ull * (uint64_t)i);
}

/* Signature classes: 0 comm (sig < 32), 1 GEMM, 2 attention, 3 elementwise. */
WL_HD uint32_t wl_sig_class(uint32_t sig) {
  if (sig < 32u) return 0u;
  uint32_t m = sig & 3u;
  return m == 0u ? 1u : (m == 1u ? 2u : 3u);
}

/* Bijection of [0, n): 4-round Feistel on the next even power of two, cycle-walked. */
WL_HD uint64_t wl_perm(uint64_t i, uint64_t n, uint64_t seed) {
  uint32_t bits = 2;
  while (((uint64_t)1 << bits) < n) bits += 2;
  const uint32_t half = bits >> 1;
  const uint64_t mask = ((uint64_t)1 << half) - 1;
  uint64_t x = i;
  do {
    uint64_t l = x >> half, r = x & mask;
    for (uint32_t k = 0; k < 4; ++k) {
      uint64_t f = wl_mix(r + seed + 0x632BE59BD9B4E019ull * (uint64_t)(k + 1)) & mask;
      uint64_t nl = r; r = l ^ f; l = nl;
    }
    x = (l << half) | r;
  } while (x >= n);
  return x;
}

WL_HD uint32_t wl_fault_mult(const wl_desc* d, uint32_t rank, uint32_t t, uint32_t sig,
                             uint32_t phase) {
  uint64_t m = 65536u;
  for (uint32_t f = d->fault_off[rank]; f < d->fault_off[rank + 1]; ++f) {
    const wl_fault* q = &d->faults[f];
    if ((q->step == 0xFFFFFFFFu || q->step == t) && (q->sig == 0xFFFFFFFFu || q->sig == sig) &&
        (q->sig_class == 0xFFFFFFFFu || q->sig_class == wl_sig_class(sig)) &&
        (q->phase == 0xFFFFFFFFu || q->phase == phase))
      m = (m * q->mult_q16) >> 16;
  }
  return (uint32_t)m;
}

/* Generate all T steps of one rank.  Event e of step t goes to out[dst(g)], g = (rank*T+t)*N+e:
 * dst(g) = g - g0 when !shuffle (rank-major order, g0 = index of the caller's first event),
 * dst(g) = wl_perm(g, R*T*N, seed) when shuffle (out is then the full buffer, g0 = 0). */
WL_HD void wl_expand_rank(const wl_desc* d, uint32_t rank, wl_event* out, uint64_t g0) {
  const uint32_t T = d->n_steps, N = d->n_events, J = d->n_streams, P = d->n_phases;
  const uint64_t total = (uint64_t)d->n_ranks * T * N;
  int64_t t0 = 1000;                       /* rank timelines start at 1 us */
  for (uint32_t t = 0; t < T; ++t) {
    const uint32_t* off = d->prog_off + (uint64_t)t * (J + 1);
    const uint32_t* prog = d->prog_sig + (uint64_t)t * N;
    uint32_t pos[WL_MAX_STREAMS];
    int64_t next_start[WL_MAX_STREAMS];
    int64_t t_end = t0;
    for (uint32_t j = 0; j < J; ++j) {
      pos[j] = 0;
      uint64_t h = wl_hash(d->seed, rank, t, j, 0);
      next_start[j] = t0 + (int64_t)d->gap_ns[(h >> 12) & 4095u];
    }
    for (uint32_t e = 0; e < N; ++e) {
      uint32_t jb = 0xFFFFFFFFu;
      int64_t best = 0;
      for (uint32_t j = 0; j < J; ++j) {
        if (pos[j] < off[j + 1] - off[j] && (jb == 0xFFFFFFFFu || next_start[j] < best)) {
          jb = j; best = next_start[j];
        }
      }
      const uint32_t i = pos[jb];
      const uint32_t sig = prog[off[jb] + i];
      const uint32_t phase = (uint32_t)(((uint64_t)e * P) / N);
      const uint64_t h = wl_hash(d->seed, rank, t, jb, i);
      uint64_t dur;
      if (d->dur_mode == 0) {
        dur = (d->base_ns[sig] * (uint64_t)d->jit_q16[h & 4095u]) >> 16;
        if (d->mode2_q16[sig] != 0u && ((h >> 47) & 1u)) dur = (dur * (uint64_t)d->mode2_q16[sig]) >> 16;
      } else {
        uint32_t i1 = (uint32_t)(h >> 24) & 65535u;
        dur = (d->xmin_ns * (uint64_t)d->pareto_q16[i1]) >> 16;
        if (i1 == 65535u) dur = (dur * (uint64_t)d->pareto_q16[(uint32_t)(h >> 40) & 65535u]) >> 16;
      }
      dur = (dur * (uint64_t)wl_fault_mult(d, rank, t, sig, phase)) >> 16;
      if (dur < 1) dur = 1;
      wl_event ev;
      ev.rank = rank; ev.step = d->step_base + t; ev.sig = sig;
      ev.stream = d->stream_id[jb]; ev.phase = (uint16_t)phase;
      ev.start_ns = best; ev.end_ns = best + (int64_t)dur;
      const uint64_t g = ((uint64_t)rank * T + t) * N + e;
      out[d->shuffle ? wl_perm(g, total, d->seed) : g - g0] = ev;
      pos[jb] = i + 1;
      if (ev.end_ns > t_end) t_end = ev.end_ns;
      const uint64_t h2 = wl_hash(d->seed, rank, t, jb, i + 1);
      next_start[jb] = ev.end_ns + (int64_t)d->gap_ns[(h2 >> 12) & 4095u];
    }
    t0 = t_end + (int64_t)d->step_gap_ns;
  }
}

#endif /* WL_EXPAND_CORE_H_ */
