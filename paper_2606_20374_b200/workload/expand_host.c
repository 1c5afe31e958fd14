/* expand_host.c — host build of the workload expander (see expand_core.h), pthreads over ranks.
 * C ABI: wl_expand_host.  Input generator only: none of the method's arithmetic lives here. */
#include "expand_core.h"
#include <pthread.h>
#include <stdlib.h>

typedef struct {
  const wl_desc* d;
  wl_event* out;
  uint32_t rank_lo, rank_hi;
  uint32_t* next;            /* shared work counter */
  pthread_mutex_t* mu;
} wl_job;

static void* wl_worker(void* p) {
  wl_job* jb = (wl_job*)p;
  const wl_desc* d = jb->d;
  const uint64_t per_rank = (uint64_t)d->n_steps * d->n_events;
  for (;;) {
    pthread_mutex_lock(jb->mu);
    uint32_t r = (*jb->next)++;
    pthread_mutex_unlock(jb->mu);
    if (r >= jb->rank_hi) break;
    if (d->shuffle) wl_expand_rank(d, r, jb->out, 0);
    else wl_expand_rank(d, r, jb->out + (uint64_t)(r - jb->rank_lo) * per_rank, (uint64_t)r * per_rank);
  }
  return 0;
}

/* Expand ranks [rank_lo, rank_hi).  !shuffle: out holds (rank_hi-rank_lo)*T*N events in
 * (rank, step, start) order.  shuffle: out is the FULL R*T*N buffer; only the given ranks'
 * events are scattered into it.  Returns 0, or -1 on bad arguments. */
int wl_expand_host(const wl_desc* d, uint32_t rank_lo, uint32_t rank_hi, wl_event* out,
                   int n_threads) {
  if (!d || !out || rank_lo > rank_hi || rank_hi > d->n_ranks || d->n_streams > WL_MAX_STREAMS ||
      d->n_streams == 0)
    return -1;
  if (n_threads < 1) n_threads = 1;
  if (n_threads > 256) n_threads = 256;
  pthread_mutex_t mu = PTHREAD_MUTEX_INITIALIZER;
  uint32_t next = rank_lo;
  wl_job job = {d, out, rank_lo, rank_hi, &next, &mu};
  pthread_t th[256];
  for (int i = 1; i < n_threads; ++i) pthread_create(&th[i], 0, wl_worker, &job);
  wl_worker(&job);
  for (int i = 1; i < n_threads; ++i) pthread_join(th[i], 0);
  return 0;
}

uint64_t wl_perm_host(uint64_t i, uint64_t n, uint64_t seed) { return wl_perm(i, n, seed); }
unsigned wl_desc_bytes(void) { return (unsigned)sizeof(wl_desc); }
