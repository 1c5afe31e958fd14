// partition.cu — grouping pass for ungrouped input (BASELINE.json configs[3]: "records shuffled
// uniformly across rank-steps, so aggregation cannot rely on contiguous segments").
//
// Folding shuffled events straight into a dense table that is far larger than L2 costs several
// random 32-byte read-modify-writes in HBM per event (aggregate_global.cu: 6 G events/s).  Moving
// each 32-byte record ONCE to its (rank, step) group costs two sequential reads (count, scatter) and
// one sector-sized write (a single 256-bit store) that L2 merges into full lines — after which the
// segmented kernel runs at streaming speed.
// Kernels, all on the caller's stream; key = rank*T + step - step_base, and
// key-invalid events go to bin R*T:
//   count   : every CTA owns a contiguous chunk of the buffer and counts its keys in a shared-memory
//             histogram (no global atomics), then writes its row H[cta][key]
//   offsets : per key, exclusive running sum over the CTAs (H[cta][key] becomes the CTA's offset
//             inside the key's group) and the group size total[key]
//   scan    : exclusive prefix sum of total in place (one CTA, running carry)
//   scatter : the same CTA re-reads its chunk with cursor[key] = total[key] + H[cta][key] in shared
//             memory: pos = atomicAdd(&cursor[key], 1); grouped[pos] = event (one 256-bit store)
// When R*T + 1 counters do not fit shared memory, count and scatter use L2 atomics on one global
// counter array instead (same results, slower).  All buffers are areas of the ctx workspace.
// Events whose key fields are out of range travel in the last bin, so that the segmented kernel
// still sees (and counts) every event; sig / phase / timestamp validity is its business.
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

}  // namespace

// CTAs of the grouping pass and whether their key histograms (R*T + 1 counters) fit shared memory.
void argus_partition_plan(const argus_config* cfg, int sm_count, int max_smem_optin, uint32_t* n_cta,
                          bool* smem) {
  const size_t bin_bytes = sizeof(uint32_t) * ((size_t)cfg->n_ranks * cfg->n_steps + 1u);
  *smem = bin_bytes <= 200u * 1024u && bin_bytes + 1024u <= (size_t)max_smem_optin;
  *n_cta = *smem ? (uint32_t)sm_count * (bin_bytes <= 100u * 1024u ? 2u : 1u) : 0u;
}

cudaError_t argus_configure_partition(argus_ctx* ctx) {
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
