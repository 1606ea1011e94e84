// reduce.cuh -- deterministic grid-wide sum: warp shuffle -> block -> per-block partial ->
// the last block to finish sums the partials in a fixed order ("warp-shuffle dot
// and norm reductions", no second kernel, no host sync, bit-reproducible for a fixed grid).
#pragma once
#include "internal.cuh"

namespace qcd {

__device__ __forceinline__ double warp_sum(double v)
{
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v += __shfl_down_sync(0xffffffffu, v, o);
    return v;
}

// Sum over the block; result valid in every thread. BLOCK multiple of 32, <= 1024.
template <int BLOCK>
__device__ __forceinline__ double block_sum(double v)
{
    __shared__ double sm[32];
    __shared__ double total;
    const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
    v = warp_sum(v);
    __syncthreads();  // protects sm/total against a previous call
    if (lane == 0) sm[wid] = v;
    __syncthreads();
    if (wid == 0) {
        double t = lane < BLOCK / 32 ? sm[lane] : 0.0;
        t = warp_sum(t);
        if (lane == 0) total = t;
    }
    __syncthreads();
    return total;
}

// Every block contributes v (already summed over its threads' work).  Returns true in ALL threads
// of the one block that finishes last, with `total` = sum over all blocks in blockIdx order.
template <int BLOCK>
__device__ __forceinline__ bool grid_sum_last_block(double v, double *partial, unsigned *counter,
                                                    double &total)
{
    __shared__ bool is_last;
    double b = block_sum<BLOCK>(v);
    if (threadIdx.x == 0) {
        partial[blockIdx.x] = b;
        __threadfence();
        unsigned ticket = atomicAdd(counter, 1u);
        is_last = (ticket == gridDim.x - 1);
    }
    __syncthreads();
    if (!is_last) return false;
    __threadfence();
    double t = 0.0;
    for (unsigned i = threadIdx.x; i < gridDim.x; i += BLOCK) t += __ldcg(partial + i);
    total = block_sum<BLOCK>(t);
    if (threadIdx.x == 0) *counter = 0u;
    return true;
}

// N block sums at once: the shuffles of the N values interleave and the block pays two barriers, not 2N.
// Each sum is formed exactly as block_sum forms it (same tree), result valid in every thread.
template <int BLOCK, int N>
__device__ __forceinline__ void block_sum_n(double (&v)[N])
{
    __shared__ double sm[N][32];
    __shared__ double total[N];
    const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
#pragma unroll
    for (int o = 16; o > 0; o >>= 1)
#pragma unroll
        for (int j = 0; j < N; ++j) v[j] += __shfl_down_sync(0xffffffffu, v[j], o);
    __syncthreads();  // protects sm/total against a previous call
    if (lane == 0)
#pragma unroll
        for (int j = 0; j < N; ++j) sm[j][wid] = v[j];
    __syncthreads();
    if (wid < N) {     // warp j finishes sum j (BLOCK / 32 >= N is asserted below)
        double t = lane < BLOCK / 32 ? sm[wid][lane] : 0.0;
        t = warp_sum(t);
        if (lane == 0) total[wid] = t;
    }
    __syncthreads();
#pragma unroll
    for (int j = 0; j < N; ++j) v[j] = total[j];
}

// N sums at once with ONE ticket: partial[blockIdx * N + j].  Returns true in all threads of the block
// that finishes last, with total[j] = sum over blocks (blockIdx order) of v[j].
template <int BLOCK, int N>
__device__ __forceinline__ bool grid_sum_last_block_n(const double (&v)[N], double *partial,
                                                      unsigned *counter, double (&total)[N])
{
    static_assert(BLOCK / 32 >= N, "block_sum_n needs one warp per sum");
    __shared__ bool is_last;
    double b[N];
#pragma unroll
    for (int j = 0; j < N; ++j) b[j] = v[j];
    block_sum_n<BLOCK, N>(b);
    if (threadIdx.x == 0) {
#pragma unroll
        for (int j = 0; j < N; ++j) partial[(size_t)blockIdx.x * N + j] = b[j];
        __threadfence();
        unsigned ticket = atomicAdd(counter, 1u);
        is_last = (ticket == gridDim.x - 1);
    }
    __syncthreads();
    if (!is_last) return false;
    __threadfence();
#pragma unroll
    for (int j = 0; j < N; ++j) {
        double t = 0.0;
        for (unsigned i = threadIdx.x; i < gridDim.x; i += BLOCK) t += __ldcg(partial + (size_t)i * N + j);
        total[j] = t;
    }
    block_sum_n<BLOCK, N>(total);
    if (threadIdx.x == 0) *counter = 0u;
    return true;
}

}  // namespace qcd
