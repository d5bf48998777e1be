// reduce.cuh -- deterministic fp64 reductions: warp shuffle tree -> shared memory ->
// one partial per block; a single-block pass adds the partials in a fixed order.
// No atomics anywhere, so the result depends only on the launch shape.
#pragma once
#include <cuda_runtime.h>

__device__ __forceinline__ double warp_sum(double v)
{
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v += __shfl_down_sync(0xffffffffu, v, o);
    return v;
}

__device__ __forceinline__ double warp_max(double v)
{
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v = fmax(v, __shfl_down_sync(0xffffffffu, v, o));
    return v;
}

// Sum of v over the block (any block shape, blockDim product a multiple of 32, <= 1024).
// Result valid in thread 0.  `slot` is shared scratch of >= 32 doubles.
__device__ __forceinline__ double block_sum(double v, double *slot)
{
    int tid = (threadIdx.z * blockDim.y + threadIdx.y) * blockDim.x + threadIdx.x;
    int nw = (blockDim.x * blockDim.y * blockDim.z + 31) >> 5;
    v = warp_sum(v);
    __syncthreads();
    if ((tid & 31) == 0) slot[tid >> 5] = v;
    __syncthreads();
    double r = 0.0;
    if (tid < 32) {
        r = tid < nw ? slot[tid] : 0.0;
        r = warp_sum(r);
    }
    return r;
}

__device__ __forceinline__ double block_max(double v, double *slot)
{
    int tid = (threadIdx.z * blockDim.y + threadIdx.y) * blockDim.x + threadIdx.x;
    int nw = (blockDim.x * blockDim.y * blockDim.z + 31) >> 5;
    v = warp_max(v);
    __syncthreads();
    if ((tid & 31) == 0) slot[tid >> 5] = v;
    __syncthreads();
    double r = -1.0e300;
    if (tid < 32) {
        r = tid < nw ? slot[tid] : -1.0e300;
        r = warp_max(r);
    }
    return r;
}

// Adds `n` partials per row for `rows` rows (row r at partials + r*stride) in a fixed
// order: thread t sums elements t, t+256, ...; then the block tree.  One block of 256.
static __global__ void finalize_sums_kernel(const double *partials, int n, int rows, int stride, double *out)
{
    __shared__ double slot[32];
    for (int r = 0; r < rows; ++r) {
        double v = 0.0;
        for (int i = threadIdx.x; i < n; i += blockDim.x) v += partials[(size_t)r * stride + i];
        double s = block_sum(v, slot);
        if (threadIdx.x == 0) out[r] = s;
        __syncthreads();
    }
}

static __global__ void finalize_max_kernel(const double *partials, int n, double *out)
{
    __shared__ double slot[32];
    double v = -1.0e300;
    for (int i = threadIdx.x; i < n; i += blockDim.x) v = fmax(v, partials[i]);
    double s = block_max(v, slot);
    if (threadIdx.x == 0) out[0] = s;
}

// Fused second stage ("last block done"): every block publishes `rows` partial sums (held by
// thread 0 in vals[]), takes an INTEGER ticket, and the block that draws the last ticket adds all
// partials -- thread t sums elements t, t+T, ... of each row, then the block tree -- and writes
// out[0..rows).  Which block is last varies from run to run, the order of the additions does not:
// the result depends on the launch shape only.  `counter` must be 0 at launch; the last block
// resets it.  All threads of the block must call this (it synchronises).  `slot`: >= 32 doubles.
template <int ROWS>
__device__ __forceinline__ void publish_and_finalize(const double (&vals)[ROWS], int rows, double *partials, int stride,
                                                     unsigned int *counter, double *out, double *slot)
{
    __shared__ int last_flag;
    const int tid = (threadIdx.z * blockDim.y + threadIdx.y) * blockDim.x + threadIdx.x;
    const int nthr = blockDim.x * blockDim.y * blockDim.z;
    const unsigned int nblk = gridDim.x * gridDim.y * gridDim.z;
    const unsigned int blk = (blockIdx.z * gridDim.y + blockIdx.y) * gridDim.x + blockIdx.x;
    if (tid == 0) {
#pragma unroll
        for (int r = 0; r < ROWS; ++r)
            if (r < rows) partials[(size_t)r * stride + blk] = vals[r];
        __threadfence();
        last_flag = (atomicAdd(counter, 1u) == nblk - 1u);
    }
    __syncthreads();
    if (!last_flag) return;
    __threadfence();
    for (int r = 0; r < rows; ++r) {
        double v = 0.0;
        for (unsigned int i = tid; i < nblk; i += nthr) v += __ldcg(partials + (size_t)r * stride + i);
        const double s = block_sum(v, slot);
        if (tid == 0) out[r] = s;
    }
    if (tid == 0) *counter = 0u;
}

// Sharded launches (fbs.cu, cbct_fbs_reconstruct_sharded): a block only publishes its partial sums at its index in the
// FULL launch's numbering; the sums are added by finalize_sums_kernel once every rank's partials are in -- in the same
// order as publish_and_finalize's last block (thread t adds elements t, t + 256, ...: both run 256 threads).
template <int ROWS>
__device__ __forceinline__ void publish_only(const double (&vals)[ROWS], int rows, double *partials, int stride, unsigned int blk)
{
    const int tid = (threadIdx.z * blockDim.y + threadIdx.y) * blockDim.x + threadIdx.x;
    if (tid == 0) {
#pragma unroll
        for (int r = 0; r < ROWS; ++r)
            if (r < rows) partials[(size_t)r * stride + blk] = vals[r];
    }
}
