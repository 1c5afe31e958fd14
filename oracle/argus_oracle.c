/* argus_oracle.c — the CPU ORACLE of the ARGUS hot path.  TEST INFRASTRUCTURE, NOT PRODUCT.
 *
 * Plain, slow, single-threaded C (fixed-width integers; no SIMD, no blocking, no fusion) of what
 * the path computes, written from the paper and the north-star text (NS = BASELINE.json
 * `north_star`; R<n> = reading n of DESIGN.md §3; PAPER.md = /root/reference/PAPER.md).
 * Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may
 * call it.  It shares no code with the CUDA path: it includes no header of include/ or of the
 * package, and re-declares the byte layouts it needs from the DESIGN.md readings.
 *
 * Every result is an exact integer function of the input multiset of records (all reductions are
 * commutative and associative; the median is an order statistic), so the oracle IS the plain
 * definition, and the CUDA path must match it byte for byte.
 *
 * Pins (tests/test_oracle_*.py, -m "not gpu"): the hand-worked example of tests/golden/
 * (SURVEY.md §8(c)), a pure-Python dict brute force, bucket() against int.bit_length at every
 * power of two +-1, closed forms of median/MAD (constant series, one outlier, arithmetic
 * progression, translation invariance, odd-R scaling), permutation and chunk-split invariance,
 * histogram/count/min/max/span invariants, recovery of the injected faults; every byte of the record
 * header (R17) by the hand-worked H lines of tests/golden/handworked.txt and a Python-int brute force
 * over the raw events (first start / last end per rank-step, zero reserved words).
 */
#include <stdint.h>
#include <stdlib.h>
#include <string.h>

/* ---- layouts (R1, R5, R17) ---------------------------------------------------------------- */
typedef struct {            /* NS: {u32 rank, u32 step, u32 sig, u16 stream, u16 phase, i64 start_ns, i64 end_ns} */
  uint32_t rank, step, sig;
  uint16_t stream, phase;
  int64_t start_ns, end_ns;
} o_event;                  /* 32 B */

typedef struct {            /* NS: count, u64 sum, min, max of duration, 32-bucket log2 histogram */
  uint64_t count, sum, min, max;
  uint32_t hist[32];
} o_cell;                   /* 160 B */

typedef struct {            /* NS: iteration / phase time = max(end) - min(start) */
  int64_t min_start, max_end;
  uint64_t span, n;
} o_span;                   /* 32 B */

typedef struct {            /* R17 header of the fixed-size per-(rank, step) record */
  uint32_t magic;
  uint16_t version, n_phases;
  uint32_t n_sigs, rank, step, reserved0;
  uint64_t n_events;
  int64_t min_start, max_end;
  uint64_t iter_ns, reserved1;
} o_header;                 /* 64 B */

typedef struct {            /* per-series output of the cross-rank rule */
  uint64_t median, mad;
  uint32_t n_high, n_low;
  uint64_t reserved;
} o_stat;                   /* 32 B */

typedef struct oracle_state {
  uint32_t R, T, S, P, step_base;
  o_cell* cells;            /* [R][T][S]   */
  o_span* spans;            /* [R][T][P+1] index P = whole iteration */
  uint64_t n_valid, n_invalid;
} oracle_state;

/* ---- R4: bucket(d) = d==0 ? 0 : min(31, floor(log2 d)).  "32-bucket log2 duration histogram"
 * (NS); the paper's log transform of durations onto an equally spaced grid.
 * Written as a shift loop on purpose (the CUDA path uses a count-leading-zeros instruction). */
uint32_t oracle_bucket(uint64_t d) {
  uint32_t b = 0;
  while (d > 1) { d >>= 1; ++b; }
  return b > 31 ? 31 : b;
}

static void cell_identity(o_cell* c) {      /* R7 */
  memset(c, 0, sizeof *c);
  c->min = UINT64_MAX;
}
static void span_identity(o_span* s) {      /* R7 */
  s->min_start = INT64_MAX; s->max_end = INT64_MIN; s->span = 0; s->n = 0;
}

oracle_state* oracle_create(uint32_t R, uint32_t T, uint32_t S, uint32_t P, uint32_t step_base) {
  oracle_state* st = (oracle_state*)calloc(1, sizeof *st);
  if (!st) return 0;
  st->R = R; st->T = T; st->S = S; st->P = P; st->step_base = step_base;
  size_t nc = (size_t)R * T * S, ns = (size_t)R * T * (P + 1);
  st->cells = (o_cell*)malloc(nc * sizeof(o_cell));
  st->spans = (o_span*)malloc(ns * sizeof(o_span));
  if (!st->cells || !st->spans) { free(st->cells); free(st->spans); free(st); return 0; }
  for (size_t i = 0; i < nc; ++i) cell_identity(&st->cells[i]);
  for (size_t i = 0; i < ns; ++i) span_identity(&st->spans[i]);
  return st;
}

void oracle_destroy(oracle_state* st) {
  if (!st) return;
  free(st->cells); free(st->spans); free(st);
}

/* ---- first half: reduce raw events (SURVEY.md §8(c) definition; PAPER.md:160-198 what it
 * stands for).  Any order, any chunking: accumulates into the state. */
void oracle_aggregate(oracle_state* st, const void* events, uint64_t n) {
  const o_event* ev = (const o_event*)events;
  for (uint64_t i = 0; i < n; ++i) {
    const o_event* e = &ev[i];
    /* R2: end < start or start < 0 -> invalid.  R3: key fields out of range -> invalid.
     * `stream` is neither validated nor used (R3, R16). */
    uint32_t t = e->step - st->step_base;            /* wraps for step < step_base -> >= T */
    if (e->start_ns < 0 || e->end_ns < e->start_ns || e->rank >= st->R || e->step < st->step_base ||
        t >= st->T || e->sig >= st->S || e->phase >= st->P) {
      st->n_invalid++;
      continue;
    }
    st->n_valid++;
    uint64_t d = (uint64_t)(e->end_ns - e->start_ns);
    o_cell* c = &st->cells[((size_t)e->rank * st->T + t) * st->S + e->sig];
    c->count += 1;
    c->sum += d;                                     /* R6: wraps mod 2^64 */
    if (d < c->min) c->min = d;
    if (d > c->max) c->max = d;
    c->hist[oracle_bucket(d)] += 1;
    /* NS span rule, for the event's phase and for the whole iteration (index P) */
    uint32_t ks[2] = { e->phase, st->P };
    for (int q = 0; q < 2; ++q) {
      o_span* s = &st->spans[((size_t)e->rank * st->T + t) * (st->P + 1) + ks[q]];
      if (e->start_ns < s->min_start) s->min_start = e->start_ns;
      if (e->end_ns > s->max_end) s->max_end = e->end_ns;
      s->n += 1;
    }
  }
}

/* span = n ? max_end - min_start : 0 for every span (NS; R8). */
void oracle_phase_times(oracle_state* st) {
  size_t ns = (size_t)st->R * st->T * (st->P + 1);
  for (size_t i = 0; i < ns; ++i) {
    o_span* s = &st->spans[i];
    s->span = s->n ? (uint64_t)(s->max_end - s->min_start) : 0;
  }
}

uint64_t oracle_record_bytes(const oracle_state* st) {
  return 64u + 32u * (uint64_t)(st->P + 1) + 160u * (uint64_t)st->S;
}

/* R17: fixed-size per-(rank, step) record = header + span[P+1] + cell[S]; table [R][T]. */
void oracle_encode_records(oracle_state* st, void* out) {
  oracle_phase_times(st);
  uint64_t rb = oracle_record_bytes(st);
  for (uint32_t r = 0; r < st->R; ++r)
    for (uint32_t t = 0; t < st->T; ++t) {
      uint8_t* p = (uint8_t*)out + ((uint64_t)r * st->T + t) * rb;
      const o_span* sp = &st->spans[((size_t)r * st->T + t) * (st->P + 1)];
      o_header h;
      memset(&h, 0, sizeof h);
      h.magic = 0x53475241u;                 /* "ARGS" */
      h.version = 1; h.n_phases = (uint16_t)st->P; h.n_sigs = st->S;
      h.rank = r; h.step = st->step_base + t;
      h.n_events = sp[st->P].n; h.min_start = sp[st->P].min_start; h.max_end = sp[st->P].max_end;
      h.iter_ns = sp[st->P].span;
      memcpy(p, &h, 64);
      memcpy(p + 64, sp, 32u * (st->P + 1));
      memcpy(p + 64 + 32u * (st->P + 1), &st->cells[((size_t)r * st->T + t) * st->S], 160u * (size_t)st->S);
    }
}

const void* oracle_cells(const oracle_state* st) { return st->cells; }
const void* oracle_spans(const oracle_state* st) { return st->spans; }
uint64_t oracle_n_valid(const oracle_state* st) { return st->n_valid; }
uint64_t oracle_n_invalid(const oracle_state* st) { return st->n_invalid; }

/* ---- second half: the cross-rank rule (NS: "per (step, sig), the exact median and MAD over
 * ranks of the u64 summed duration and flags a rank when |x - median| > 3*MAD, all in integer
 * arithmetic"; the paper's cross-rank comparison of the same kernel). */
static int cmp_u64(const void* a, const void* b) {
  uint64_t x = *(const uint64_t*)a, y = *(const uint64_t*)b;
  return x < y ? -1 : (x > y ? 1 : 0);
}

/* R10: median = lo + (hi - lo)/2 with lo = v[(R-1)/2], hi = v[R/2] of the sorted series. */
static uint64_t median_u64(const uint64_t* x, uint32_t R, uint64_t* tmp) {
  memcpy(tmp, x, (size_t)R * 8);
  qsort(tmp, R, 8, cmp_u64);
  uint64_t lo = tmp[(R - 1) / 2], hi = tmp[R / 2];
  return lo + (hi - lo) / 2;
}

/* One series of R values -> stat + flags[R].  Exposed for the closed-form pins. */
void oracle_series(const uint64_t* x, uint32_t R, o_stat* stat, uint8_t* flags) {
  uint64_t* tmp = (uint64_t*)malloc((size_t)R * 8);
  uint64_t* dev = (uint64_t*)malloc((size_t)R * 8);
  uint64_t med = median_u64(x, R, tmp);
  for (uint32_t r = 0; r < R; ++r) dev[r] = x[r] >= med ? x[r] - med : med - x[r];
  uint64_t mad = median_u64(dev, R, tmp);
  uint64_t thr = mad > UINT64_MAX / 3 ? UINT64_MAX : 3 * mad;        /* R12 saturating 3*MAD */
  uint32_t nh = 0, nl = 0;
  for (uint32_t r = 0; r < R; ++r) {
    uint8_t f = 0;
    if (dev[r] > thr) f = x[r] > med ? 1 : 2;                          /* R13 strict >, R14 direction */
    if (f == 1) nh++;
    if (f == 2) nl++;
    if (flags) flags[r] = f;
  }
  stat->median = med; stat->mad = mad; stat->n_high = nh; stat->n_low = nl; stat->reserved = 0;
  free(tmp); free(dev);
}

/* All series of the table (R11: all R ranks, empty cell counts as x = 0; R15: same rule on the
 * phase spans and the whole-iteration span, plus the roll-ups).  Any output may be NULL. */
void oracle_diagnose(oracle_state* st, o_stat* sig_stats /*[T][S]*/, uint8_t* sig_flags /*[T][S][R]*/,
                     o_stat* span_stats /*[T][P+1]*/, uint8_t* span_flags /*[T][P+1][R]*/,
                     uint32_t* rank_score /*[T][R]*/, uint32_t* step_anomalous /*[T]*/) {
  oracle_phase_times(st);
  const uint32_t R = st->R, T = st->T, S = st->S, P = st->P;
  uint64_t* x = (uint64_t*)malloc((size_t)R * 8);
  uint8_t* fl = (uint8_t*)malloc(R);
  if (rank_score) memset(rank_score, 0, (size_t)T * R * 4);
  if (step_anomalous) memset(step_anomalous, 0, (size_t)T * 4);
  for (uint32_t t = 0; t < T; ++t) {
    for (uint32_t s = 0; s < S; ++s) {
      for (uint32_t r = 0; r < R; ++r) {
        const o_cell* c = &st->cells[((size_t)r * T + t) * S + s];
        x[r] = c->count ? c->sum : 0;
      }
      o_stat stt;
      oracle_series(x, R, &stt, fl);
      if (sig_stats) sig_stats[(size_t)t * S + s] = stt;
      if (sig_flags) memcpy(sig_flags + ((size_t)t * S + s) * R, fl, R);
      if (rank_score)
        for (uint32_t r = 0; r < R; ++r) rank_score[(size_t)t * R + r] += fl[r] == 1;
    }
    for (uint32_t k = 0; k <= P; ++k) {
      for (uint32_t r = 0; r < R; ++r) x[r] = st->spans[((size_t)r * T + t) * (P + 1) + k].span;
      o_stat stt;
      oracle_series(x, R, &stt, fl);
      if (span_stats) span_stats[(size_t)t * (P + 1) + k] = stt;
      if (span_flags) memcpy(span_flags + ((size_t)t * (P + 1) + k) * R, fl, R);
      if (k == P && step_anomalous) step_anomalous[t] = stt.n_high;
    }
  }
  free(x); free(fl);
}
