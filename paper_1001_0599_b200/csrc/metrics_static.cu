// metrics_static.cu -- cbct_quality_metrics_static: the image-quality metrics of metrics.cu (PAPER.md:L263,
//     e = ||f - f0||_2 / ||f0||_2,   c = corr(f, f0))
// for callers that cannot allocate (code under CUDA graph capture, tight serving loops, harnesses that forbid cudaMalloc).
// cbct_quality_metrics needs a cbct_geometry handle, whose creation allocates the reduction scratch (block partials, ticket,
// pinned host mirror).  This entry point needs no handle and calls no cudaMalloc / cudaFree / allocating routine: its scratch is
// the file-scope array below, which every GPU that loads the library holds until the process exits.
//
// Scratch: CBCT_STATIC_MAX_BLOCKS x 6 fp64 block partials + one 256-byte line for the ticket = 786 688 bytes.  A block sums a
// FIXED chunk of CBCT_STATIC_CHUNK consecutive elements, so the number of blocks -- and the order of every addition -- depends
// on n alone (not on the device's SM count), and n is bounded by CBCT_STATIC_MAX_ELEMS = 2^28 elements (1 GiB per volume;
// config 4 is 2^26).  Larger volumes are refused with CBCT_ERR_INVALID_ARG.
//
// EVERY call shares the array and it keeps the last call's contents: the partials are all overwritten before they are read;
// the ticket must start at zero and is cleared on the caller's stream before every launch (a call that died half-way cannot
// poison the next).  Two calls that overlap on the GPU (different streams, or two host threads) race on it: callers serialise.
#include <mutex>
#include "cbct_internal.cuh"
#include "reduce.cuh"

constexpr int MS_THREADS = 256, MS_PER_THREAD = 64;
constexpr int MS_CHUNK = MS_THREADS * MS_PER_THREAD;                      // 16 384 elements per block
constexpr int MS_MAX_BLOCKS = 16384;
constexpr unsigned long long MS_MAX_ELEMS = (unsigned long long)MS_CHUNK * MS_MAX_BLOCKS;   // 2^28
constexpr int MS_TICKET_AT = 6 * MS_MAX_BLOCKS;                           // the ticket's line, in doubles from the start
static_assert(MS_CHUNK == CBCT_STATIC_CHUNK && MS_MAX_BLOCKS == CBCT_STATIC_MAX_BLOCKS && MS_MAX_ELEMS == CBCT_STATIC_MAX_ELEMS,
              "include/cbct.h states these limits");

// In HOST code this name is a host-side stand-in, not a device address: the kernel is given the pointer that
// cudaGetSymbolAddress returns for the current device (static_scratch()).
static __device__ __align__(256) double cbct_static_scratch[6 * MS_MAX_BLOCKS + 32];

// partials[r * MS_MAX_BLOCKS + b]: sum r of block b; out2 = (e, c), written by the block that draws the last ticket, which adds
// the partials in block order (thread t: blocks t, t + 256, ...; then the block tree) -- the scheme of reduce.cuh.
__global__ void __launch_bounds__(MS_THREADS)
quality_metrics_static_kernel(unsigned long long n, const float *__restrict__ f, const float *__restrict__ f0,
                              double *__restrict__ scratch, double *__restrict__ out2)
{
    __shared__ double slot[32];
    __shared__ int last_flag;
    const unsigned long long base = (unsigned long long)blockIdx.x * MS_CHUNK;
    double s[6] = {0.0, 0.0, 0.0, 0.0, 0.0, 0.0};
#pragma unroll 4
    for (int i = 0; i < MS_PER_THREAD; ++i) {
        const unsigned long long o = base + (unsigned long long)i * MS_THREADS + threadIdx.x;
        if (o < n) {
            const double a = (double)__ldg(f + o), b = (double)__ldg(f0 + o), d = a - b;
            s[0] += a; s[1] += b;
            s[2] = fma(a, a, s[2]); s[3] = fma(b, b, s[3]); s[4] = fma(a, b, s[4]); s[5] = fma(d, d, s[5]);
        }
    }
    double v[6];
#pragma unroll
    for (int r = 0; r < 6; ++r) v[r] = block_sum(s[r], slot);
    unsigned int *ticket = reinterpret_cast<unsigned int *>(scratch + MS_TICKET_AT);
    if (threadIdx.x == 0) {
#pragma unroll
        for (int r = 0; r < 6; ++r) scratch[(size_t)r * MS_MAX_BLOCKS + blockIdx.x] = v[r];
        __threadfence();
        last_flag = (atomicAdd(ticket, 1u) == gridDim.x - 1u);
    }
    __syncthreads();
    if (!last_flag) return;
    __threadfence();
    double h[6];
    for (int r = 0; r < 6; ++r) {
        double p = 0.0;
        for (unsigned int i = threadIdx.x; i < gridDim.x; i += MS_THREADS) p += __ldcg(scratch + (size_t)r * MS_MAX_BLOCKS + i);
        h[r] = block_sum(p, slot);
    }
    if (threadIdx.x == 0) {
        // the arithmetic of cbct_quality_metrics (metrics.cu), on the device: 0 for a metric whose denominator vanishes
        const double nn = (double)n;
        out2[0] = h[3] > 0.0 ? sqrt(h[5] / h[3]) : 0.0;
        const double cov = h[4] - h[0] * h[1] / nn, va = h[2] - h[0] * h[0] / nn, vb = h[3] - h[1] * h[1] / nn;
        out2[1] = (va > 0.0 && vb > 0.0) ? cov / sqrt(va * vb) : 0.0;
        *ticket = 0u;
    }
}

// Device address of the scratch array on the CURRENT device; looked up once per device (set-up), with that device current.
static cbct_status static_scratch(double **out)
{
    constexpr int MAX_DEV = 64;
    static std::mutex mtx;
    static double *addr[MAX_DEV] = {nullptr};
    int dev = -1;
    CBCT_CUDA(cudaGetDevice(&dev));
    if (dev < 0 || dev >= MAX_DEV) return cbct_fail(CBCT_ERR_UNSUPPORTED, "cbct_quality_metrics_static: device ordinal %d out of range", dev);
    std::lock_guard<std::mutex> lock(mtx);
    if (!addr[dev]) {
        void *p = nullptr;
        CBCT_CUDA(cudaGetSymbolAddress(&p, cbct_static_scratch));
        if (!p) return cbct_fail(CBCT_ERR_CUDA, "cbct_quality_metrics_static: cudaGetSymbolAddress returned NULL");
        addr[dev] = static_cast<double *>(p);
    }
    *out = addr[dev];
    return CBCT_OK;
}

extern "C" cbct_status cbct_quality_metrics_static(const float *d_f, const float *d_f0, unsigned long long n,
                                                   double *d_out2, void *cuda_stream)
{
    if (!d_f || !d_f0 || !d_out2) return cbct_fail(CBCT_ERR_INVALID_ARG, "cbct_quality_metrics_static: NULL buffer");
    if (n == 0) return cbct_fail(CBCT_ERR_INVALID_ARG, "cbct_quality_metrics_static: n = 0");
    if (n > MS_MAX_ELEMS)
        return cbct_fail(CBCT_ERR_INVALID_ARG, "cbct_quality_metrics_static: n = %llu exceeds the static scratch's maximum of %llu "
                         "elements (CBCT_STATIC_MAX_ELEMS); use cbct_quality_metrics", n, MS_MAX_ELEMS);
    cudaStream_t st = (cudaStream_t)cuda_stream;
    double *scratch = nullptr;
    cbct_status s = static_scratch(&scratch);
    if (s != CBCT_OK) return s;
    const unsigned int blocks = (unsigned int)((n + MS_CHUNK - 1) / MS_CHUNK);
    CBCT_CUDA(cudaMemsetAsync(scratch + MS_TICKET_AT, 0, 256, st));       // the ticket starts at zero, whatever the last call left
    quality_metrics_static_kernel<<<blocks, MS_THREADS, 0, st>>>(n, d_f, d_f0, scratch, d_out2);
    cudaError_t e = cudaGetLastError();
    if (e != cudaSuccess) return cbct_fail(CBCT_ERR_CUDA, "cbct_quality_metrics_static: kernel launch: %s", cudaGetErrorString(e));
    return CBCT_OK;
}
