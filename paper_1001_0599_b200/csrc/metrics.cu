// metrics.cu -- NEXT-3 of the scope table: the paper's two image-quality metrics, the relative
// error  e = ||f - f0||_2 / ||f0||_2  and the correlation coefficient  c = corr(f, f0)  between a reconstruction
// f and the ground truth f0, as ONE fused pass over both volumes: six fp64 sums (f, f0, f^2, f0^2, f f0,
// (f - f0)^2) per thread, fixed-order block and grid reduction (reduce.cuh), the last block forms e and c.
// HBM bound: 8 bytes per voxel.
#include "cbct_internal.cuh"
#include "reduce.cuh"

constexpr int MET_BLOCKS_PER_SM = 4, MET_THREADS = 256;

__global__ void __launch_bounds__(MET_THREADS)
quality_metrics_kernel(size_t n, const float *__restrict__ f, const float *__restrict__ f0, double *__restrict__ partials,
                       unsigned int *__restrict__ counter, double *__restrict__ out)
{
    __shared__ double slot[32];
    double s[6] = {0.0, 0.0, 0.0, 0.0, 0.0, 0.0};
    for (size_t o = (size_t)blockIdx.x * blockDim.x + threadIdx.x; o < n; o += (size_t)gridDim.x * blockDim.x) {
        const double a = (double)__ldg(f + o), b = (double)__ldg(f0 + o), d = a - b;
        s[0] += a; s[1] += b;
        s[2] = fma(a, a, s[2]); s[3] = fma(b, b, s[3]); s[4] = fma(a, b, s[4]); s[5] = fma(d, d, s[5]);
    }
    double v[6];
#pragma unroll
    for (int r = 0; r < 6; ++r) v[r] = block_sum(s[r], slot);
    publish_and_finalize<6>(v, 6, partials, (int)gridDim.x, counter, out, slot);
}

static cbct_status six_sums(const cbct_geometry *g, size_t n, const float *d_a, const float *d_b, cudaStream_t st)
{
    int blocks = g->sm_count * MET_BLOCKS_PER_SM;
    if ((size_t)blocks * 6 > (size_t)4 * g->partials_stride) blocks = 4 * g->partials_stride / 6;
    {
        StageTimer t(g, st, ST_REDUCE);
        quality_metrics_kernel<<<blocks, MET_THREADS, 0, st>>>(n, d_a, d_b, g->d_partials, g->d_counter, g->d_scalars);
        CBCT_LAUNCH_CHECK(g);
    }
    CBCT_CUDA(cudaMemcpyAsync(g->h_scalars, g->d_scalars, 6 * sizeof(double), cudaMemcpyDeviceToHost, st));
    CBCT_CUDA(cudaStreamSynchronize(st));
    return CBCT_OK;
}

cbct_status volume_change(const cbct_geometry *g, size_t n, const float *d_a, const float *d_b, double *sum_d2,
                          double *sum_b2, cudaStream_t st)
{
    cbct_status s = six_sums(g, n, d_a, d_b, st);
    if (s != CBCT_OK) return s;
    *sum_d2 = g->h_scalars[5];
    *sum_b2 = g->h_scalars[3];
    return CBCT_OK;
}

// the six sums come back to the host, which forms e and c from them (a handful of fp64 flops)
extern "C" cbct_status cbct_quality_metrics(const cbct_geometry *g, int level, const float *d_f, const float *d_f0,
                                            double *rel_error, double *correlation, void *cuda_stream)
{
    const Level *L = get_level(g, level);
    if (!L || !d_f || !d_f0 || !rel_error || !correlation)
        return cbct_fail(CBCT_ERR_INVALID_ARG, "cbct_quality_metrics: bad handle, level or NULL");
    cbct_status s = six_sums(g, L->nvox, d_f, d_f0, (cudaStream_t)cuda_stream);
    if (s != CBCT_OK) return s;
    const double *h = g->h_scalars, n = (double)L->nvox;
    *rel_error = h[3] > 0.0 ? sqrt(h[5] / h[3]) : 0.0;
    const double cov = h[4] - h[0] * h[1] / n, va = h[2] - h[0] * h[0] / n, vb = h[3] - h[1] * h[1] / n;
    *correlation = (va > 0.0 && vb > 0.0) ? cov / sqrt(va * vb) : 0.0;
    return CBCT_OK;
}
