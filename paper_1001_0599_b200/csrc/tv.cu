// tv.cu -- A6/A7/A9: the ROF / TV-prox sub-solver of Algorithm A1 step 2 and the
// non-negativity truncation of step 3.
//
//   E_ROF[f] = mean_v |grad f|_delta + (beta/2) mean_v (f - g)^2        (L151, L155; S6)
//   d        = N_vox dE_ROF/df = -div p + beta (f - g),  p = grad f / |grad f|_delta
//   Armijo (Eq. 5; S10):  E[f - s d] <= E0 - c s mean(d^2), else s <- alpha s
// Forward differences in mm^-1; neighbour outside the grid = 0 (BC_ZERO) or the voxel's own
// value (BC_REFLECT) (L161).  div is the exact negative transpose (backward differences,
// p_{-1} = 0).  Per-voxel terms are fp32, sums are fp64 in a fixed order (reduce.cuh).
#include <math.h>
#include "cbct_internal.cuh"
#include "reduce.cuh"

struct TvDims {
    int nx, ny, nz;
    float ihx, ihy, ihz;   // 1/h
    int zero_xy, zero_z;   // 1 = BC_ZERO
};

static TvDims tv_dims(const Level &L)
{
    TvDims D;
    D.nx = L.p.nx; D.ny = L.p.ny; D.nz = L.p.nz;
    D.ihx = (float)(1.0 / L.hx); D.ihy = (float)(1.0 / L.hy); D.ihz = (float)(1.0 / L.hz);
    D.zero_xy = L.p.bc_xy == CBCT_BC_ZERO; D.zero_z = L.p.bc_z == CBCT_BC_ZERO;
    return D;
}

// forward-difference gradient at (i,j,k) of the field  f - lam*d  (d may be NULL)
template <bool TRIAL>
__device__ __forceinline__ float field(const float *__restrict__ f, const float *__restrict__ d, float lam, size_t o)
{
    return TRIAL ? fmaf(-lam, __ldg(d + o), __ldg(f + o)) : __ldg(f + o);
}

template <bool TRIAL>
__device__ __forceinline__ void grad3(const TvDims &D, const float *__restrict__ f, const float *__restrict__ d,
                                      float lam, int i, int j, int k, float &c, float &gx, float &gy, float &gz)
{
    const size_t o = ((size_t)k * D.ny + j) * D.nx + i;
    c = field<TRIAL>(f, d, lam, o);
    const float xn = (i + 1 < D.nx) ? field<TRIAL>(f, d, lam, o + 1) : (D.zero_xy ? 0.0f : c);
    const float yn = (j + 1 < D.ny) ? field<TRIAL>(f, d, lam, o + D.nx) : (D.zero_xy ? 0.0f : c);
    const float zn = (k + 1 < D.nz) ? field<TRIAL>(f, d, lam, o + (size_t)D.nx * D.ny) : (D.zero_z ? 0.0f : c);
    gx = (xn - c) * D.ihx; gy = (yn - c) * D.ihy; gz = (zn - c) * D.ihz;
}

constexpr int TV_BX = 32, TV_BY = 4, TV_BZ = 2;

// partial sums, row 0: sum |grad f|_delta, row 1: sum (f-g)^2, row 2: sum d^2 (GRAD only)
// GRAD: also writes d.   TRIAL: evaluates the field f - lam*dir instead of f.
template <bool GRAD, bool TRIAL>
__global__ void __launch_bounds__(TV_BX *TV_BY *TV_BZ)
tv_pass_kernel(const TvDims D, const float *__restrict__ f, const float *__restrict__ dir,
               const float *__restrict__ g, const double *__restrict__ lam_ptr, float beta, float delta2,
               float *__restrict__ d_out, double *__restrict__ partials, int stride)
{
    __shared__ double slot[32];
    const int i = blockIdx.x * TV_BX + threadIdx.x;
    const int j = blockIdx.y * TV_BY + threadIdx.y;
    const int k = blockIdx.z * TV_BZ + threadIdx.z;
    const float lam = TRIAL ? (float)lam_ptr[0] : 0.0f;
    double e_tv = 0.0, e_q = 0.0, e_d = 0.0;
    if (i < D.nx && j < D.ny && k < D.nz) {
        float c, gx, gy, gz;
        grad3<TRIAL>(D, f, dir, lam, i, j, k, c, gx, gy, gz);
        const float nrm2 = fmaf(gx, gx, fmaf(gy, gy, fmaf(gz, gz, delta2)));
        const float nrm = sqrtf(nrm2);
        e_tv = nrm;
        const size_t o = ((size_t)k * D.ny + j) * D.nx + i;
        const float r = g ? c - __ldg(g + o) : 0.0f;
        e_q = (double)r * r;
        if (GRAD) {
            const float inv = 1.0f / nrm;
            float div = (gx * D.ihx + gy * D.ihy + gz * D.ihz) * inv;
            float c2, ax, ay, az;
            if (i > 0) {
                grad3<false>(D, f, nullptr, 0.f, i - 1, j, k, c2, ax, ay, az);
                div -= ax * D.ihx * rsqrtf(fmaf(ax, ax, fmaf(ay, ay, fmaf(az, az, delta2))));
            }
            if (j > 0) {
                grad3<false>(D, f, nullptr, 0.f, i, j - 1, k, c2, ax, ay, az);
                div -= ay * D.ihy * rsqrtf(fmaf(ax, ax, fmaf(ay, ay, fmaf(az, az, delta2))));
            }
            if (k > 0) {
                grad3<false>(D, f, nullptr, 0.f, i, j, k - 1, c2, ax, ay, az);
                div -= az * D.ihz * rsqrtf(fmaf(ax, ax, fmaf(ay, ay, fmaf(az, az, delta2))));
            }
            const float dd = fmaf(beta, r, -div);
            d_out[o] = dd;
            e_d = (double)dd * dd;
        }
    }
    const int blk = (blockIdx.z * gridDim.y + blockIdx.y) * gridDim.x + blockIdx.x;
    double s0 = block_sum(e_tv, slot);
    if (threadIdx.x == 0 && threadIdx.y == 0 && threadIdx.z == 0) partials[blk] = s0;
    double s1 = block_sum(e_q, slot);
    if (threadIdx.x == 0 && threadIdx.y == 0 && threadIdx.z == 0) partials[stride + blk] = s1;
    if (GRAD) {
        double s2 = block_sum(e_d, slot);
        if (threadIdx.x == 0 && threadIdx.y == 0 && threadIdx.z == 0) partials[2 * stride + blk] = s2;
    }
}

// f_out = f - lam * d  (optionally clipped at 0: Algorithm A1 step 3, L149)
__global__ void tv_update_kernel(size_t n, const float *__restrict__ f, const float *__restrict__ d,
                                 const double *__restrict__ lam_ptr, int clip, float *__restrict__ out)
{
    const float lam = (float)lam_ptr[0];
    for (size_t o = (size_t)blockIdx.x * blockDim.x + threadIdx.x; o < n; o += (size_t)gridDim.x * blockDim.x) {
        float v = fmaf(-lam, d[o], f[o]);
        out[o] = (clip && v < 0.0f) ? 0.0f : v;
    }
}

__global__ void clip_copy_kernel(size_t n, const float *__restrict__ in, int clip, float *__restrict__ out)
{
    for (size_t o = (size_t)blockIdx.x * blockDim.x + threadIdx.x; o < n; o += (size_t)gridDim.x * blockDim.x) {
        float v = in[o];
        out[o] = (clip && v < 0.0f) ? 0.0f : v;
    }
}

static dim3 tv_grid(const TvDims &D)
{
    return dim3((D.nx + TV_BX - 1) / TV_BX, (D.ny + TV_BY - 1) / TV_BY, (D.nz + TV_BZ - 1) / TV_BZ);
}

cbct_status launch_tv_energy(const cbct_geometry *g, const Level &L, const float *d_f, double delta,
                             double *d_out, cudaStream_t st)
{
    TvDims D = tv_dims(L);
    dim3 gr = tv_grid(D), b(TV_BX, TV_BY, TV_BZ);
    const int nblk = gr.x * gr.y * gr.z;
    if (nblk > g->partials_stride) return cbct_fail(CBCT_ERR_INVALID_ARG, "volume too large for the reduction buffer");
    StageTimer t(g, st, ST_REDUCE);
    tv_pass_kernel<false, false><<<gr, b, 0, st>>>(D, d_f, nullptr, nullptr, nullptr, 0.f, (float)(delta * delta),
                                                  nullptr, g->d_partials, g->partials_stride);
    CBCT_LAUNCH_CHECK(g);
    finalize_sums_kernel<<<1, 256, 0, st>>>(g->d_partials, nblk, 1, g->partials_stride, d_out);
    CBCT_LAUNCH_CHECK(g);
    return CBCT_OK;
}

// Host-driven control loop: every trial reads two fp64 sums back (one stream sync per
// pass).  Scalars: d_scalars[0..2] = sums, d_scalars[4] = trial step.
cbct_status run_tv_prox(const cbct_geometry *g, const Level &L, const float *d_g, float *d_f, double w,
                        int nonneg, const cbct_tv_params &tp, cbct_tv_report *rep, bool sync_report,
                        cudaStream_t st)
{
    (void)sync_report;
    cbct_tv_report r = {0, 0, 0.0, 0.0};
    const size_t n = L.nvox;
    const int cp_blocks = g->sm_count * 8;
    if (w <= 0.0) {
        StageTimer t(g, st, ST_TV_UPDATE);
        clip_copy_kernel<<<cp_blocks, 256, 0, st>>>(n, d_g, nonneg, d_f);
        CBCT_LAUNCH_CHECK(g);
        if (rep) *rep = r;
        return CBCT_OK;
    }
    TvDims D = tv_dims(L);
    dim3 gr = tv_grid(D), b(TV_BX, TV_BY, TV_BZ);
    const int nblk = gr.x * gr.y * gr.z, S = g->partials_stride;
    if (nblk > S) return cbct_fail(CBCT_ERR_INVALID_ARG, "volume too large for the reduction buffer");
    const double beta = 1.0 / w, N = (double)n;
    const float delta2 = (float)(tp.eps_delta * tp.eps_delta);
    double *ds = g->d_scalars, *hs = g->h_scalars;
    // ping-pong: cur holds f; the first f is g itself (read-only), later ones alternate
    const float *cur = d_g;
    float *bufs[2] = {d_f, L.d_f2};
    int which = 0;
    double E0 = 0.0;
    bool have_E0 = false;
    for (int it = 0; it < tp.max_inner; ++it) {
        {
            StageTimer t(g, st, ST_TV_GRAD);
            tv_pass_kernel<true, false><<<gr, b, 0, st>>>(D, cur, nullptr, d_g, nullptr, (float)beta, delta2, L.d_d,
                                                         g->d_partials, S);
            CBCT_LAUNCH_CHECK(g);
        }
        {
            StageTimer t(g, st, ST_REDUCE);
            finalize_sums_kernel<<<1, 256, 0, st>>>(g->d_partials, nblk, 3, S, ds);
            CBCT_LAUNCH_CHECK(g);
        }
        CBCT_CUDA(cudaMemcpyAsync(hs, ds, 3 * sizeof(double), cudaMemcpyDeviceToHost, st));
        CBCT_CUDA(cudaStreamSynchronize(st));
        if (!have_E0) { E0 = hs[0] / N + 0.5 * beta * hs[1] / N; r.e_first = r.e_last = E0; have_E0 = true; }
        const double Dm = hs[2] / N;
        double lam = 1.0 / beta, Enew = E0;
        bool accepted = false;
        for (int bt = 0; bt <= tp.max_backtracks; ++bt) {
            hs[4] = lam;
            CBCT_CUDA(cudaMemcpyAsync(ds + 4, hs + 4, sizeof(double), cudaMemcpyHostToDevice, st));
            {
                StageTimer t(g, st, ST_TV_TRIAL);
                tv_pass_kernel<false, true><<<gr, b, 0, st>>>(D, cur, L.d_d, d_g, ds + 4, (float)beta, delta2, nullptr,
                                                             g->d_partials, S);
                CBCT_LAUNCH_CHECK(g);
            }
            {
                StageTimer t(g, st, ST_REDUCE);
                finalize_sums_kernel<<<1, 256, 0, st>>>(g->d_partials, nblk, 2, S, ds);
                CBCT_LAUNCH_CHECK(g);
            }
            CBCT_CUDA(cudaMemcpyAsync(hs, ds, 2 * sizeof(double), cudaMemcpyDeviceToHost, st));
            CBCT_CUDA(cudaStreamSynchronize(st));
            Enew = hs[0] / N + 0.5 * beta * hs[1] / N;
            ++r.trials;
            if (Enew <= E0 - tp.armijo_c * lam * Dm) { accepted = true; break; }
            lam *= tp.shrink_alpha;
        }
        if (!accepted) break;
        float *nxt = bufs[which];
        which ^= 1;
        {
            StageTimer t(g, st, ST_TV_UPDATE);
            tv_update_kernel<<<cp_blocks, 256, 0, st>>>(n, cur, L.d_d, ds + 4, 0, nxt);
            CBCT_LAUNCH_CHECK(g);
        }
        cur = nxt;
        ++r.inner_iters;
        const double rel = fabs(Enew - E0) / E0;
        E0 = Enew;
        r.e_last = Enew;
        if (rel < tp.rel_tol) break;
    }
    // result to d_f, with the non-negativity truncation
    if (cur != d_f || nonneg) {
        StageTimer t(g, st, ST_TV_UPDATE);
        clip_copy_kernel<<<cp_blocks, 256, 0, st>>>(n, cur, nonneg, d_f);
        CBCT_LAUNCH_CHECK(g);
    }
    if (rep) *rep = r;
    return CBCT_OK;
}

extern "C" cbct_status cbct_tv_prox(const cbct_geometry *g, int level, const float *d_g, float *d_f,
                                    double weight_w, int nonneg, const cbct_tv_params *params,
                                    cbct_tv_report *report, void *cuda_stream)
{
    const Level *L = get_level(g, level);
    if (!L || !d_g || !d_f || !params || d_g == d_f)
        return cbct_fail(CBCT_ERR_INVALID_ARG, "cbct_tv_prox: bad handle, level, NULL or aliased buffer");
    if (!(weight_w >= 0.0) || params->max_inner < 0 || params->max_backtracks < 0 ||
        !(params->shrink_alpha > 0.0 && params->shrink_alpha < 1.0))
        return cbct_fail(CBCT_ERR_INVALID_ARG, "cbct_tv_prox: bad parameter");
    cudaStream_t st = (cudaStream_t)cuda_stream;
    cbct_status s = run_tv_prox(g, *L, d_g, d_f, weight_w, nonneg, *params, report, true, st);
    if (s == CBCT_OK && report) CBCT_CUDA(cudaStreamSynchronize(st));
    return s;
}

extern "C" cbct_status cbct_tv_energy(const cbct_geometry *g, int level, const float *d_f, double eps_delta,
                                      double *e1, void *cuda_stream)
{
    const Level *L = get_level(g, level);
    if (!L || !d_f || !e1) return cbct_fail(CBCT_ERR_INVALID_ARG, "cbct_tv_energy: bad handle, level or NULL");
    cudaStream_t st = (cudaStream_t)cuda_stream;
    cbct_status s = launch_tv_energy(g, *L, d_f, eps_delta, g->d_scalars + 8, st);
    if (s != CBCT_OK) return s;
    CBCT_CUDA(cudaMemcpyAsync(g->h_scalars + 8, g->d_scalars + 8, sizeof(double), cudaMemcpyDeviceToHost, st));
    CBCT_CUDA(cudaStreamSynchronize(st));
    *e1 = g->h_scalars[8] / (double)L->nvox;
    return CBCT_OK;
}
