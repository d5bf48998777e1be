// transfer.cu -- A8: multi-grid transfers (readings S12, S13) and a few
// element-wise helpers.  All HBM-bound, one thread per output element.
#include "cbct_internal.cuh"
#include "reduce.cuh"

// coarse[k][j][i] = mean of the 2x2x2 fine block
// A pair of x-neighbours: one 8-byte load when the caller's buffer is 8-byte aligned (VEC), two 4-byte loads otherwise
// (a torch view at an odd element offset); the row length is even, so every pair of an aligned buffer is aligned.
template <bool VEC>
__device__ __forceinline__ float2 load_pair(const float *__restrict__ p)
{
    if (VEC) return __ldg(reinterpret_cast<const float2 *>(p));
    return make_float2(__ldg(p), __ldg(p + 1));
}

template <bool VEC>
__global__ void restrict_kernel(int cx, int cy, int cz, const float *__restrict__ fine, float *__restrict__ coarse)
{
    const int i = blockIdx.x * blockDim.x + threadIdx.x, j = blockIdx.y * blockDim.y + threadIdx.y, k = blockIdx.z;
    if (i >= cx || j >= cy) return;
    const int nx = 2 * cx, ny = 2 * cy;
    float s = 0.0f;
#pragma unroll
    for (int c = 0; c < 2; ++c)
#pragma unroll
        for (int b = 0; b < 2; ++b) {
            const float2 v = load_pair<VEC>(fine + ((size_t)(2 * k + c) * ny + (2 * j + b)) * nx + 2 * i);
            s += v.x + v.y;
        }
    coarse[((size_t)k * cy + j) * cx + i] = 0.125f * s;
}

// coarse[a][j][i] = mean of the 2x2 fine pixels
template <bool VEC>
__global__ void bin_kernel(int cu, int cv, const float *__restrict__ fine, float *__restrict__ coarse)
{
    const int i = blockIdx.x * blockDim.x + threadIdx.x, j = blockIdx.y * blockDim.y + threadIdx.y, a = blockIdx.z;
    if (i >= cu || j >= cv) return;
    const int nu = 2 * cu, nv = 2 * cv;
    const float2 r0 = load_pair<VEC>(fine + ((size_t)a * nv + 2 * j) * nu + 2 * i);
    const float2 r1 = load_pair<VEC>(fine + ((size_t)a * nv + 2 * j + 1) * nu + 2 * i);
    coarse[((size_t)a * cv + j) * cu + i] = 0.25f * ((r0.x + r0.y) + (r1.x + r1.y));
}

// Cell-centred trilinear prolongation (reading S13).  Along one axis a fine cell n lies between the centres of the
// coarse cells lo = floor((n - 1) / 2) and lo + 1, a quarter of a coarse cell from the nearer one: the nearer cell -- lo + 1
// for even n, lo for odd n -- weighs 3/4.  A cell outside the grid counts 0 (BC_ZERO) or repeats the edge cell (BC_REFLECT).
struct ProlongTap {
    int lo, hi;         // clamped indices of the two coarse cells
    float wlo, whi;     // their weights, 0 for a cell that counts as 0
};

__device__ __forceinline__ ProlongTap prolong_tap(int n, int nc, bool zero_outside)
{
    ProlongTap t;
    const int lo = (n - 1) >> 1;                    // arithmetic shift: -1 for n = 0
    const bool even = (n & 1) == 0;
    t.wlo = even ? 0.25f : 0.75f;
    t.whi = even ? 0.75f : 0.25f;
    if (zero_outside && lo < 0) t.wlo = 0.0f;
    if (zero_outside && lo + 1 >= nc) t.whi = 0.0f;
    t.lo = max(lo, 0);
    t.hi = min(lo + 1, nc - 1);
    return t;
}

__global__ void prolong_kernel(int cx, int cy, int cz, int zero_xy, int zero_z,
                               const float *__restrict__ coarse, float *__restrict__ fine)
{
    const int i = blockIdx.x * blockDim.x + threadIdx.x, j = blockIdx.y * blockDim.y + threadIdx.y, k = blockIdx.z;
    const int nx = 2 * cx, ny = 2 * cy;
    if (i >= nx || j >= ny) return;
    const ProlongTap tx = prolong_tap(i, cx, zero_xy != 0), ty = prolong_tap(j, cy, zero_xy != 0), tz = prolong_tap(k, cz, zero_z != 0);
    const float *p00 = coarse + ((size_t)tz.lo * cy + ty.lo) * cx, *p01 = coarse + ((size_t)tz.lo * cy + ty.hi) * cx;
    const float *p10 = coarse + ((size_t)tz.hi * cy + ty.lo) * cx, *p11 = coarse + ((size_t)tz.hi * cy + ty.hi) * cx;
    // x first, then y, then z
    const float r00 = tx.wlo * __ldg(p00 + tx.lo) + tx.whi * __ldg(p00 + tx.hi);
    const float r01 = tx.wlo * __ldg(p01 + tx.lo) + tx.whi * __ldg(p01 + tx.hi);
    const float r10 = tx.wlo * __ldg(p10 + tx.lo) + tx.whi * __ldg(p10 + tx.hi);
    const float r11 = tx.wlo * __ldg(p11 + tx.lo) + tx.whi * __ldg(p11 + tx.hi);
    const float s0 = ty.wlo * r00 + ty.whi * r01, s1 = ty.wlo * r10 + ty.whi * r11;
    fine[((size_t)k * ny + j) * nx + i] = tz.wlo * s0 + tz.whi * s1;
}

__global__ void max_kernel(size_t n, const float *__restrict__ x, double *__restrict__ partials)
{
    __shared__ double slot[32];
    double m = -1.0e300;
    for (size_t o = (size_t)blockIdx.x * blockDim.x + threadIdx.x; o < n; o += (size_t)gridDim.x * blockDim.x)
        m = fmax(m, (double)x[o]);
    double r = block_max(m, slot);
    if (threadIdx.x == 0) partials[blockIdx.x] = r;
}

__global__ void fill_kernel(size_t n, float val, float *__restrict__ x)
{
    for (size_t o = (size_t)blockIdx.x * blockDim.x + threadIdx.x; o < n; o += (size_t)gridDim.x * blockDim.x) x[o] = val;
}

cbct_status launch_restrict(const cbct_geometry *g, const Level &fine, const float *d_fine, float *d_coarse, cudaStream_t st)
{
    const int cx = fine.p.nx / 2, cy = fine.p.ny / 2, cz = fine.p.nz / 2;
    dim3 b(32, 8), gr((cx + 31) / 32, (cy + 7) / 8, cz);
    StageTimer t(g, st, ST_TRANSFER);
    if ((uintptr_t)d_fine % 8 == 0) restrict_kernel<true><<<gr, b, 0, st>>>(cx, cy, cz, d_fine, d_coarse);
    else restrict_kernel<false><<<gr, b, 0, st>>>(cx, cy, cz, d_fine, d_coarse);
    CBCT_LAUNCH_CHECK(g);
    return CBCT_OK;
}

cbct_status launch_bin(const cbct_geometry *g, const Level &fine, const float *d_fine, float *d_coarse, cudaStream_t st)
{
    const int cu = fine.p.nu / 2, cv = fine.p.nv / 2;
    dim3 b(32, 8), gr((cu + 31) / 32, (cv + 7) / 8, fine.p.np);
    StageTimer t(g, st, ST_TRANSFER);
    if ((uintptr_t)d_fine % 8 == 0) bin_kernel<true><<<gr, b, 0, st>>>(cu, cv, d_fine, d_coarse);
    else bin_kernel<false><<<gr, b, 0, st>>>(cu, cv, d_fine, d_coarse);
    CBCT_LAUNCH_CHECK(g);
    return CBCT_OK;
}

cbct_status launch_prolong(const cbct_geometry *g, const Level &fine, const float *d_coarse, float *d_fine, cudaStream_t st)
{
    const int cx = fine.p.nx / 2, cy = fine.p.ny / 2, cz = fine.p.nz / 2;
    dim3 b(32, 8), gr((fine.p.nx + 31) / 32, (fine.p.ny + 7) / 8, fine.p.nz);
    StageTimer t(g, st, ST_TRANSFER);
    prolong_kernel<<<gr, b, 0, st>>>(cx, cy, cz, fine.p.bc_xy == CBCT_BC_ZERO, fine.p.bc_z == CBCT_BC_ZERO, d_coarse, d_fine);
    CBCT_LAUNCH_CHECK(g);
    return CBCT_OK;
}

cbct_status launch_max(const cbct_geometry *g, const float *d_x, size_t n, double *d_out, cudaStream_t st)
{
    const int blocks = 1024 < g->partials_stride ? 1024 : g->partials_stride;
    StageTimer t(g, st, ST_TRANSFER);
    max_kernel<<<blocks, 256, 0, st>>>(n, d_x, g->d_partials);
    CBCT_LAUNCH_CHECK(g);
    finalize_max_kernel<<<1, 256, 0, st>>>(g->d_partials, blocks, d_out);
    CBCT_LAUNCH_CHECK(g);
    return CBCT_OK;
}

cbct_status launch_fill(const cbct_geometry *g, float *d_x, size_t n, float val, cudaStream_t st)
{
    StageTimer t(g, st, ST_TRANSFER);
    fill_kernel<<<g->sm_count * 8, 256, 0, st>>>(n, val, d_x);
    CBCT_LAUNCH_CHECK(g);
    return CBCT_OK;
}

static const Level *fine_of_pair(const cbct_geometry *g, int level)
{
    if (!g || level < 0 || level + 1 >= (int)g->levels.size()) return nullptr;
    return &g->levels[level];
}

extern "C" cbct_status cbct_restrict_volume(const cbct_geometry *g, int level, const float *d_fine, float *d_coarse, void *cuda_stream)
{
    const Level *L = fine_of_pair(g, level);
    if (!L || !d_fine || !d_coarse) return cbct_fail(CBCT_ERR_INVALID_ARG, "cbct_restrict_volume: level+1 must be a provisioned level; buffers non-NULL");
    return launch_restrict(g, *L, d_fine, d_coarse, (cudaStream_t)cuda_stream);
}

extern "C" cbct_status cbct_bin_projections(const cbct_geometry *g, int level, const float *d_fine, float *d_coarse, void *cuda_stream)
{
    const Level *L = fine_of_pair(g, level);
    if (!L || !d_fine || !d_coarse) return cbct_fail(CBCT_ERR_INVALID_ARG, "cbct_bin_projections: level+1 must be a provisioned level; buffers non-NULL");
    return launch_bin(g, *L, d_fine, d_coarse, (cudaStream_t)cuda_stream);
}

extern "C" cbct_status cbct_prolong_volume(const cbct_geometry *g, int level, const float *d_coarse, float *d_fine, void *cuda_stream)
{
    const Level *L = fine_of_pair(g, level);
    if (!L || !d_fine || !d_coarse) return cbct_fail(CBCT_ERR_INVALID_ARG, "cbct_prolong_volume: level+1 must be a provisioned level; buffers non-NULL");
    return launch_prolong(g, *L, d_coarse, d_fine, (cudaStream_t)cuda_stream);
}
