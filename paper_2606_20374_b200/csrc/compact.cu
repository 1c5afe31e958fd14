// compact.cu — the compact record encodings (second half: "sparse/bit-packed record
// encoding (non-empty bins only) to raise the compression ratio"; the paper's record of "approximately 200
// triples ... about 2.7 KB").  Two variable-length encodings of a finalised table, both a
// stream compaction (DESIGN.md §3 R37, R38; byte layouts in include/argus.h):
//   SPARSE  lossless: header, the non-empty phase spans, and per non-empty cell {sig, b0, nb, count, sum,
//           min, max, hist[b0 .. b0 + nb)} — only the histogram buckets between bucket(min) and bucket(max)
//   TRIPLE  the paper's: header, spans, and per cell with clusters {sig, n, n x (count, p50_bin, p99_bin)}
// One kernel on the caller's stream, one CTA per record: the CTA sizes its record (the 32-byte head of every
// cell, or one byte of d_n_clusters), learns its offset in the stream by a decoupled look-back over the records
// before it, and writes header, spans, then the cells in tiles of one sig per thread, each tile placed by a
// block-wide exclusive scan of its entry sizes — the table is read once.  (Tables whose per-sig words do not
// fit shared memory take three kernels instead: size, scan, write.)  HBM-bound.
#include "argus_internal.cuh"

namespace {

constexpr int NT = 256;

struct Src {
  const uint8_t* records;
  const argus_cluster* clusters;   // TRIPLE: [R*T][S][mc]
  const uint8_t* n_clusters;       // TRIPLE: [R*T][S]
  uint32_t mc;
};

__device__ __forceinline__ uint32_t bucket_u64(unsigned long long d) { return argus_bucket64(d); }

// 16 bytes of a cell head.  The sizing loop reads one 32-byte sector of every 160-byte cell: ask L2 for 64-byte
// fills instead of whole 128-byte lines (every line of the table holds part of some head).
__device__ __forceinline__ unsigned long long ld64_sparse(const unsigned long long* p) {
  unsigned long long v;
  asm volatile("ld.global.nc.L2::64B.u64 %0, [%1];" : "=l"(v) : "l"(p));
  return v;
}
__device__ __forceinline__ uint32_t ld32_sparse(const uint32_t* p) {
  uint32_t v;
  asm volatile("ld.global.nc.L2::64B.u32 %0, [%1];" : "=r"(v) : "l"(p));
  return v;
}
__device__ __forceinline__ uint4 ld_head(const uint4* p) {
  uint4 v;
  asm volatile("ld.global.nc.L2::64B.v4.u32 {%0, %1, %2, %3}, [%4];" : "=r"(v.x), "=r"(v.y), "=r"(v.z), "=r"(v.w) : "l"(p));
  return v;
}

// bytes of the entry of cell (key, sig); 0 = the cell is left out.  SPARSE: also returns b0 / nb.
template <bool TRIPLE>
__device__ __forceinline__ uint32_t entry_bytes(const Src& src, const argus_dims& D, uint32_t key, uint32_t sig,
                                                uint32_t& b0, uint32_t& nb) {
  if (TRIPLE) {
    uint32_t n = src.n_clusters[(size_t)key * D.S + sig];
    n = n < src.mc ? n : src.mc;                 // a count beyond the slots of the cell cannot be honoured (and would not fit s_info)
    nb = n; b0 = 0u;
    return n ? 8u + 8u * n : 0u;
  }
  const uint4* c = reinterpret_cast<const uint4*>(src.records + (size_t)key * D.rec_bytes + D.cell_off + (size_t)sig * 160u);
  const uint4 h0 = ld_head(c);                 // {count, sum}
  if ((h0.x | h0.y) == 0u) { b0 = nb = 0u; return 0u; }
  const uint4 h1 = ld_head(c + 1);             // {min, max}
  b0 = bucket_u64(((unsigned long long)h1.y << 32) | h1.x);
  nb = bucket_u64(((unsigned long long)h1.w << 32) | h1.z) - b0 + 1u;
  return 40u + 4u * (nb + (nb & 1u));
}

// exclusive block scan of one u32 per thread (NT threads); returns the prefix, total in `total`
__device__ __forceinline__ uint32_t block_exscan(uint32_t v, uint32_t* s_warp, uint32_t& total) {
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  uint32_t inc = v;
#pragma unroll
  for (int o = 1; o < 32; o <<= 1) {
    const uint32_t t = __shfl_up_sync(0xFFFFFFFFu, inc, o);
    if (lane >= o) inc += t;
  }
  if (lane == 31) s_warp[warp] = inc;
  __syncthreads();
  uint32_t before = 0u, all = 0u;
#pragma unroll
  for (int w = 0; w < NT / 32; ++w) {
    const uint32_t x = s_warp[w];
    if (w < warp) before += x;
    all += x;
  }
  __syncthreads();                             // s_warp may be reused by the caller's next tile
  total = all;
  return before + inc - v;
}

// phase part of a record: mask of the non-empty phase spans (bit k: span[k].n_events != 0) — P <= 64
__device__ __forceinline__ unsigned long long phase_mask(const uint8_t* rec, const argus_dims& D) {
  unsigned long long m = 0ull;
  const argus_span* sp = reinterpret_cast<const argus_span*>(rec + D.span_off);
  for (uint32_t k = 0; k < D.P; ++k)
    if (sp[k].n_events != 0ull) m |= 1ull << k;
  return m;
}

template <bool TRIPLE>
__global__ void __launch_bounds__(NT)
compact_size_kernel(Src src, argus_dims D, unsigned long long* __restrict__ sizes) {
  __shared__ uint32_t s_warp[NT / 32];
  const uint32_t key = blockIdx.x;
  uint32_t bytes = 0u;
  for (uint32_t sig = threadIdx.x; sig < D.S; sig += NT) {
    uint32_t b0, nb;
    bytes += entry_bytes<TRIPLE>(src, D, key, sig, b0, nb);
  }
  uint32_t total;
  block_exscan(bytes, s_warp, total);
  if (threadIdx.x == 0) {
    const unsigned long long m = phase_mask(src.records + (size_t)key * D.rec_bytes, D);
    sizes[key] = 64ull + 8ull + 32ull * (unsigned long long)__popcll(m) + total;
  }
}

// in place: sizes[0..m) -> exclusive prefix, sizes[m] = total (one CTA)
__global__ void __launch_bounds__(1024)
compact_scan_kernel(unsigned long long* v, uint32_t m) {
  __shared__ unsigned long long s_warp[32];
  __shared__ unsigned long long s_carry;
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  if (tid == 0) s_carry = 0ull;
  __syncthreads();
  for (uint32_t base = 0; base < m; base += 1024u) {
    const uint32_t i = base + (uint32_t)tid;
    const unsigned long long x = i < m ? v[i] : 0ull;
    unsigned long long inc = x;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
      const unsigned long long t = __shfl_up_sync(0xFFFFFFFFu, inc, o);
      if (lane >= o) inc += t;
    }
    if (lane == 31) s_warp[warp] = inc;
    __syncthreads();
    unsigned long long before = 0ull, all = 0ull;
    for (int w = 0; w < 32; ++w) {
      const unsigned long long y = s_warp[w];
      if (w < warp) before += y;
      all += y;
    }
    const unsigned long long carry = s_carry;
    if (i < m) v[i] = carry + before + inc - x;
    __syncthreads();
    if (tid == 0) s_carry = carry + all;
    __syncthreads();
  }
  if (tid == 0) v[m] = s_carry;
}

__device__ __forceinline__ void st64(uint8_t* p, unsigned long long v) { *reinterpret_cast<unsigned long long*>(p) = v; }

template <bool TRIPLE>
__global__ void __launch_bounds__(NT)
compact_write_kernel(Src src, argus_dims D, const unsigned long long* __restrict__ offsets, uint8_t* __restrict__ out,
                     unsigned long long capacity) {
  __shared__ uint32_t s_warp[NT / 32];
  const uint32_t key = blockIdx.x;
  const unsigned long long beg = offsets[key], end = offsets[key + 1];
  if (end > capacity) return;                  // does not fit: the caller sees offsets[R*T] > capacity
  const uint8_t* rec = src.records + (size_t)key * D.rec_bytes;
  uint8_t* dst = out + beg;
  const unsigned long long m = phase_mask(rec, D);
  // non-empty spans, ascending k: thread k copies span k to slot popc(m & (2^k - 1))
  for (uint32_t k = threadIdx.x; k < D.P; k += NT) {
    if (m >> k & 1ull) {
      const uint4* sp = reinterpret_cast<const uint4*>(rec + D.span_off + 32u * k);
      uint4* d = reinterpret_cast<uint4*>(dst + 72u + 32u * (uint32_t)__popcll(m & ((1ull << k) - 1ull)));
      // dst + 72 is 8-byte aligned only: two 64-bit stores per half
      const uint4 a = sp[0], b = sp[1];
      unsigned long long* q = reinterpret_cast<unsigned long long*>(d);
      q[0] = ((unsigned long long)a.y << 32) | a.x; q[1] = ((unsigned long long)a.w << 32) | a.z;
      q[2] = ((unsigned long long)b.y << 32) | b.x; q[3] = ((unsigned long long)b.w << 32) | b.z;
    }
  }
  uint32_t run = 72u + 32u * (uint32_t)__popcll(m);   // bytes written so far (block-uniform)
  uint32_t n_cells = 0u;
  for (uint32_t s0 = 0; s0 < D.S; s0 += NT) {
    const uint32_t sig = s0 + threadIdx.x;
    uint32_t b0 = 0u, nb = 0u, bytes = 0u;
    if (sig < D.S) bytes = entry_bytes<TRIPLE>(src, D, key, sig, b0, nb);
    uint32_t total;
    const uint32_t pre = block_exscan(bytes, s_warp, total);
    n_cells += __syncthreads_count(bytes != 0u);
    if (bytes) {
      uint8_t* e = dst + run + pre;
      if (TRIPLE) {
        st64(e, ((unsigned long long)nb << 32) | sig);
        const unsigned long long* cl = reinterpret_cast<const unsigned long long*>(src.clusters + ((size_t)key * D.S + sig) * src.mc);
        for (uint32_t j = 0; j < nb; ++j) st64(e + 8u + 8u * j, cl[j]);
      } else {
        const unsigned long long* c = reinterpret_cast<const unsigned long long*>(rec + D.cell_off + (size_t)sig * 160u);
        st64(e, (unsigned long long)sig | ((unsigned long long)b0 << 32) | ((unsigned long long)nb << 40));
        st64(e + 8, c[0]); st64(e + 16, c[1]); st64(e + 24, c[2]); st64(e + 32, c[3]);
        const uint32_t* h = reinterpret_cast<const uint32_t*>(c + 4) + b0;
        for (uint32_t j = 0; j < nb; j += 2u) {
          const unsigned long long lo = h[j], hi = j + 1u < nb ? h[j + 1u] : 0u;
          st64(e + 40u + 4u * j, lo | (hi << 32));
        }
      }
    }
    run += total;
  }
  if (threadIdx.x == 0) {
    // header as R17 with version 2 / 3, reserved0 = cells kept, reserved1 = length
    const argus_record_header* h = reinterpret_cast<const argus_record_header*>(rec);
    argus_record_header o = *h;
    o.version = TRIPLE ? 3 : 2;
    o.reserved0 = n_cells;
    o.reserved1 = end - beg;
    const unsigned long long* q = reinterpret_cast<const unsigned long long*>(&o);
    for (int i = 0; i < 8; ++i) st64(dst + 8 * i, q[i]);
    st64(dst + 64, m);
  }
}

// ---- one pass instead of three -------------------------------------------------------------------------------
// A record's place in the stream is the sum of the sizes of the records before it.  Instead of a size pass over
// the whole table, a scan and a write pass (the table read twice), every CTA sizes its record, gets its offset by
// a DECOUPLED LOOK-BACK over the records before it, and writes — the cell heads it sized are still in L1 / L2
// when the write loop comes back for the rest of the cell.  Records are handed out by a ticket counter, so the
// CTAs a look-back waits for have started before it (forward progress).  d_offsets[k + 1] carries the state of
// record k while the kernel runs — top two bits: 1 = the size of record k alone, 2 = the inclusive prefix through
// record k — and a last small kernel strips the bits.
constexpr unsigned long long LB_AGG = 1ull << 62, LB_PRE = 2ull << 62, LB_VAL = (1ull << 62) - 1ull;
__device__ __forceinline__ unsigned long long ld_vol(const unsigned long long* p) {
  return *reinterpret_cast<const volatile unsigned long long*>(p);
}

template <bool TRIPLE>
__global__ void __launch_bounds__(NT)
compact_fused_kernel(Src src, argus_dims D, unsigned long long* offsets, uint32_t* ticket, uint8_t* __restrict__ out,
                     unsigned long long capacity) {
  extern __shared__ uint32_t s_info[];         // per sig: bytes | b0 << 8 | nb << 16
  __shared__ uint32_t s_warp[NT / 32];
  __shared__ uint32_t s_key;
  __shared__ unsigned long long s_beg;
  if (threadIdx.x == 0) s_key = atomicAdd(ticket, 1u);
  __syncthreads();
  const uint32_t key = s_key;
  if (key == 0u && threadIdx.x == 0) offsets[0] = LB_PRE;        // nothing before record 0
  const uint8_t* rec = src.records + (size_t)key * D.rec_bytes;
  // size of this record
  uint32_t bytes = 0u;
  for (uint32_t sig = threadIdx.x; sig < D.S; sig += NT) {
    uint32_t b0, nb;
    const uint32_t e = entry_bytes<TRIPLE>(src, D, key, sig, b0, nb);
    s_info[sig] = e | (b0 << 8) | (nb << 16);
    bytes += e;
  }
  uint32_t cells_bytes;
  block_exscan(bytes, s_warp, cells_bytes);
  const unsigned long long m = phase_mask(rec, D);              // every thread: a few cached loads
  const unsigned long long size = 64ull + 8ull + 32ull * (unsigned long long)__popcll(m) + cells_bytes;
  if (threadIdx.x < 32) {
    const int lane = threadIdx.x;
    if (lane == 0) atomicExch(&offsets[key + 1u], LB_AGG | size);
    // look back from slot `key` (the state of record key - 1) towards slot 0, 32 slots at a time
    unsigned long long excl = 0ull;
    long long pos = (long long)key;
    for (;;) {
      const long long i = pos - lane;
      unsigned long long v = LB_PRE;                            // below slot 0: an empty prefix
      if (i >= 0) { do { v = ld_vol(offsets + i); } while ((v >> 62) == 0ull); }
      const uint32_t pm = __ballot_sync(0xFFFFFFFFu, (v >> 62) == 2ull);
      const int f = pm ? __ffs((int)pm) - 1 : 32;               // nearest slot that holds a prefix
      unsigned long long part = lane <= f ? (v & LB_VAL) : 0ull;
#pragma unroll
      for (int o = 16; o > 0; o >>= 1) part += __shfl_xor_sync(0xFFFFFFFFu, part, o);
      excl += part;
      if (pm) break;
      pos -= 32;
    }
    if (lane == 0) {
      atomicExch(&offsets[key + 1u], LB_PRE | (excl + size));
      s_beg = excl;
    }
  }
  __syncthreads();
  const unsigned long long beg = s_beg;
  if (beg + size > capacity) return;           // does not fit: the caller sees offsets[R*T] > capacity
  uint8_t* dst = out + beg;
  for (uint32_t k = threadIdx.x; k < D.P; k += NT) {
    if (m >> k & 1ull) {
      const uint4* sp = reinterpret_cast<const uint4*>(rec + D.span_off + 32u * k);
      unsigned long long* q = reinterpret_cast<unsigned long long*>(dst + 72u + 32u * (uint32_t)__popcll(m & ((1ull << k) - 1ull)));
      const uint4 a = sp[0], b = sp[1];
      q[0] = ((unsigned long long)a.y << 32) | a.x; q[1] = ((unsigned long long)a.w << 32) | a.z;
      q[2] = ((unsigned long long)b.y << 32) | b.x; q[3] = ((unsigned long long)b.w << 32) | b.z;
    }
  }
  uint32_t run = 72u + 32u * (uint32_t)__popcll(m);
  uint32_t n_cells = 0u;
  for (uint32_t s0 = 0; s0 < D.S; s0 += NT) {
    const uint32_t sig = s0 + threadIdx.x;
    const uint32_t info = sig < D.S ? s_info[sig] : 0u;
    const uint32_t eb = info & 0xFFu, b0 = (info >> 8) & 0xFFu, nb = info >> 16;
    uint32_t total;
    const uint32_t pre = block_exscan(eb, s_warp, total);
    n_cells += __syncthreads_count(eb != 0u);
    if (eb) {
      uint8_t* e = dst + run + pre;
      if (TRIPLE) {
        st64(e, ((unsigned long long)nb << 32) | sig);
        const unsigned long long* cl = reinterpret_cast<const unsigned long long*>(src.clusters + ((size_t)key * D.S + sig) * src.mc);
        for (uint32_t j = 0; j < nb; ++j) st64(e + 8u + 8u * j, cl[j]);
      } else {
        const unsigned long long* c = reinterpret_cast<const unsigned long long*>(rec + D.cell_off + (size_t)sig * 160u);
        st64(e, (unsigned long long)sig | ((unsigned long long)b0 << 32) | ((unsigned long long)nb << 40));
        st64(e + 8, ld64_sparse(c)); st64(e + 16, ld64_sparse(c + 1)); st64(e + 24, ld64_sparse(c + 2)); st64(e + 32, ld64_sparse(c + 3));
        const uint32_t* h = reinterpret_cast<const uint32_t*>(c + 4) + b0;
        for (uint32_t j = 0; j < nb; j += 2u) {
          const unsigned long long lo = ld32_sparse(h + j), hi = j + 1u < nb ? ld32_sparse(h + j + 1u) : 0u;
          st64(e + 40u + 4u * j, lo | (hi << 32));
        }
      }
    }
    run += total;
  }
  if (threadIdx.x == 0) {
    const argus_record_header* h = reinterpret_cast<const argus_record_header*>(rec);
    argus_record_header o = *h;
    o.version = TRIPLE ? 3 : 2;
    o.reserved0 = n_cells;
    o.reserved1 = size;
    const unsigned long long* q = reinterpret_cast<const unsigned long long*>(&o);
    for (int i = 0; i < 8; ++i) st64(dst + 8 * i, q[i]);
    st64(dst + 64, m);
  }
}

__global__ void __launch_bounds__(256)
compact_strip_kernel(unsigned long long* offsets, uint32_t m) {
  const uint32_t i = blockIdx.x * blockDim.x + threadIdx.x;
  if (i <= m) offsets[i] &= LB_VAL;
}

template <bool TRIPLE>
cudaError_t launch(argus_ctx* ctx, const Src& src, uint8_t* d_out, uint64_t capacity, unsigned long long* d_offsets,
                   cudaStream_t s) {
  const uint32_t n_rec = ctx->dims.R * ctx->dims.T;
  const size_t info_bytes = sizeof(uint32_t) * (size_t)ctx->dims.S;
  // entry sizes must fit a byte (TRIPLE: 8 + 8 * max_clusters <= 136) and the per-sig words shared memory
  if (info_bytes <= 160u * 1024u && (size_t)ctx->max_smem_optin >= info_bytes + 4096u && (!TRIPLE || src.mc <= 16u)) {
    uint32_t* ticket = reinterpret_cast<uint32_t*>(ctx->d_counters + 8);    // spare word of the counters area
    cudaError_t e = cudaMemsetAsync(ticket, 0, sizeof(uint32_t), s);
    if (e == cudaSuccess) e = cudaMemsetAsync(d_offsets, 0, sizeof(unsigned long long) * ((size_t)n_rec + 1u), s);
    if (e != cudaSuccess) return e;              // (the kernel's shared-memory opt-in was set in argus_create)
    compact_fused_kernel<TRIPLE><<<n_rec, NT, info_bytes, s>>>(src, ctx->dims, d_offsets, ticket, d_out, capacity);
    compact_strip_kernel<<<(n_rec + 256u) / 256u, 256, 0, s>>>(d_offsets, n_rec);
    ctx->n_memsets += 2;
    ctx->n_kernels += 2;
    return cudaGetLastError();
  }
  compact_size_kernel<TRIPLE><<<n_rec, NT, 0, s>>>(src, ctx->dims, d_offsets);
  compact_scan_kernel<<<1, 1024, 0, s>>>(d_offsets, n_rec);
  compact_write_kernel<TRIPLE><<<n_rec, NT, 0, s>>>(src, ctx->dims, d_offsets, d_out, capacity);
  ctx->n_kernels += 3;
  return cudaGetLastError();
}

}  // namespace

cudaError_t argus_configure_compact(argus_ctx* ctx) {
  cudaError_t e = argus_optin_all_smem(compact_fused_kernel<false>, ctx->max_smem_optin);
  return e == cudaSuccess ? argus_optin_all_smem(compact_fused_kernel<true>, ctx->max_smem_optin) : e;
}

cudaError_t argus_launch_sparse_encode(argus_ctx* ctx, const void* d_records, uint8_t* d_out, uint64_t capacity,
                                       uint64_t* d_offsets, cudaStream_t s) {
  Src src{static_cast<const uint8_t*>(d_records), nullptr, nullptr, 0u};
  return launch<false>(ctx, src, d_out, capacity, reinterpret_cast<unsigned long long*>(d_offsets), s);
}

cudaError_t argus_launch_triple_encode(argus_ctx* ctx, const void* d_records, const argus_cluster* d_clusters,
                                       const uint8_t* d_n_clusters, uint32_t mc, uint8_t* d_out, uint64_t capacity,
                                       uint64_t* d_offsets, cudaStream_t s) {
  Src src{static_cast<const uint8_t*>(d_records), d_clusters, d_n_clusters, mc};
  return launch<true>(ctx, src, d_out, capacity, reinterpret_cast<unsigned long long*>(d_offsets), s);
}
