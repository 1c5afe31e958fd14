// partition.cu — grouping pass for ungrouped input (BASELINE.json configs[3]: "records shuffled
// uniformly across rank-steps, so aggregation cannot rely on contiguous segments").
//
// Folding shuffled events straight into a dense table that is far larger than L2 costs several
// random 32-byte read-modify-writes in HBM per event (aggregate_global.cu: 6 G events/s).  Moving
// each 32-byte record ONCE to its (rank, step) group costs one sequential read, one sector-sized
// write that L2 merges into full lines (one open line per group), and one L2 atomic on a counter
// array that stays L2-resident — after which the segmented kernel runs at streaming speed.
// Three kernels, all on the caller's stream:
//   count   : hist[key]++ per event (key = rank*T + step - step_base; key-invalid events -> bin R*T)
//   scan    : exclusive prefix sum of hist in place (one CTA, running carry)
//   scatter : pos = atomicAdd(&hist[key], 1); grouped[pos] = event
// Events whose key fields are out of range travel in the last bin, so that the segmented kernel
// still sees (and counts) every event; sig / phase / timestamp validity is its business.
#include "argus_internal.cuh"

namespace {

__device__ __forceinline__ uint32_t group_key(const argus_dims& D, uint32_t rank, uint32_t step) {
  const uint32_t t = step - D.step_base;
  return (rank < D.R && t < D.T) ? rank * D.T + t : D.R * D.T;
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
    grouped[2 * (size_t)pos] = lo;
    grouped[2 * (size_t)pos + 1] = hi;
  }
}

}  // namespace

// Group n events by (rank, step) into ctx->d_group (grown on demand).  Returns cudaErrorMemoryAllocation
// if the workspace cannot be had (the caller then falls back to the global-table kernel).
cudaError_t argus_launch_partition(argus_ctx* ctx, const argus_event* ev, uint64_t n, cudaStream_t s) {
  const argus_dims& D = ctx->dims;
  const uint32_t m = D.R * D.T + 1u;
  if (ctx->group_capacity < n) {
    // grow-only; the old buffer may still be read by work queued on a stream: drain first
    cudaError_t e = cudaDeviceSynchronize();
    if (e != cudaSuccess) return e;
    if (ctx->d_group) cudaFree(ctx->d_group);
    ctx->d_group = nullptr; ctx->group_capacity = 0;
    e = cudaMalloc(&ctx->d_group, n * sizeof(argus_event));
    if (e != cudaSuccess) { (void)cudaGetLastError(); return cudaErrorMemoryAllocation; }
    ctx->group_capacity = n;
  }
  cudaError_t e = cudaMemsetAsync(ctx->d_hist, 0, sizeof(uint32_t) * m, s);
  if (e != cudaSuccess) return e;
  const uint4* src = reinterpret_cast<const uint4*>(ev);
  uint64_t blocks = (n + 511) / 512;
  const uint64_t cap = (uint64_t)ctx->sm_count * 4 * 8;   // 4 CTAs of 512 per SM, a few tiles each
  if (blocks > cap) blocks = cap;
  partition_count_kernel<<<(unsigned)blocks, 512, 0, s>>>(src, n, D, ctx->d_hist);
  partition_scan_kernel<<<1, 1024, 0, s>>>(ctx->d_hist, m);
  partition_scatter_kernel<<<(unsigned)blocks, 512, 0, s>>>(src, n, D, ctx->d_hist,
                                                            reinterpret_cast<uint4*>(ctx->d_group));
  return cudaGetLastError();
}
