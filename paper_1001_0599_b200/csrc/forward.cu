// forward.cu -- A1/A2: cone-beam forward projector, one thread per detector ray.
//
// (P f)[ray] = sum_voxels len(ray ∩ voxel) f[voxel]   (Eq. 1 on piecewise-
// constant voxels; "a ray-tracing algorithm, such as Siddon's", L187, L243).
//
// Instead of Siddon's data-dependent merge of three crossing lists, the ray is cut into
// unit slabs of its DRIVING axis (the in-plane axis along which it crosses more planes).
// Inside one slab it crosses at most one plane of the other in-plane axis and at most one
// z-plane (checked at create), so it touches at most three voxels whose lengths follow in
// closed form from the two crossing parameters.  The lengths are the exact radiological
// path -- the same numbers as Siddon's up to rounding -- but every thread of a warp runs
// the same loop with the same trip structure, and neighbouring rays read neighbouring
// addresses: x-driven rays read the [k][i][j] copy of the volume, y-driven rays the
// [k][j][i] original, so the minor in-plane index is always the fastest one in memory.
#include "cbct_internal.cuh"
#include "ray.cuh"
#include "reduce.cuh"

// [k][j][i] -> [k][i][j], 32x32 tiles through shared memory
__global__ void transpose_xy_kernel(const float *__restrict__ in, float *__restrict__ out, int nx, int ny)
{
    __shared__ float tile[32][33];
    const size_t slice = (size_t)blockIdx.z * nx * ny;
    int i = blockIdx.x * 32 + threadIdx.x, j0 = blockIdx.y * 32;
    for (int r = threadIdx.y; r < 32; r += blockDim.y) {
        int j = j0 + r;
        if (i < nx && j < ny) tile[r][threadIdx.x] = __ldg(in + slice + (size_t)j * nx + i);
    }
    __syncthreads();
    int j = j0 + threadIdx.x, i0 = blockIdx.x * 32;
    for (int r = threadIdx.y; r < 32; r += blockDim.y) {
        int ii = i0 + r;
        if (ii < nx && j < ny) out[slice + (size_t)ii * ny + j] = tile[threadIdx.x][r];
    }
}

constexpr int FWD_BX = 32, FWD_BY = 8;

template <int MODE>
__global__ void __launch_bounds__(FWD_BX *FWD_BY)
forward_kernel(const LevelParams P, const float *__restrict__ vol, const float *__restrict__ volT,
               const RayU *__restrict__ rayu, const float *__restrict__ y, float *__restrict__ out,
               double *__restrict__ partials)
{
    __shared__ double slot[32];
    const int iu = blockIdx.x * FWD_BX + threadIdx.x;
    const int iv = blockIdx.y * FWD_BY + threadIdx.y;
    const int a = blockIdx.z;
    double sq = 0.0;
    if (iu < P.nu && iv < P.nv) {
        const RayU r = load_rayu(rayu, a * P.nu + iu);
        const float v = fmaf((float)iv, P.dv, P.v0);
        const RayZ rz = ray_z(r, v, P.sz);
        // driving axis: nd slabs, minor axis: nm voxels; memory index (k*nd + slab)*nm + minor
        const float *__restrict__ base = r.drive ? vol : volT;
        const int nd = r.drive ? P.ny : P.nx, nm = r.drive ? P.nx : P.ny;
        const int cd = r.drive ? P.cy : P.cx, cm = r.drive ? P.cx : P.cy;
        // slab range in which the ray can be inside the minor and z extents (conservative)
        float dlo = (float)(-cd), dhi = (float)(nd - cd);
        {
            float mlo = (float)(-cm), mhi = (float)(nm - cm);
            if (r.m != 0.0f) {
                float t1 = (mlo - r.a0) * r.inv_m, t2 = (mhi - r.a0) * r.inv_m;
                dlo = fmaxf(dlo, fminf(t1, t2) - 1.0f); dhi = fminf(dhi, fmaxf(t1, t2) + 1.0f);
            } else if (r.a0 < mlo || r.a0 >= mhi) dhi = dlo - 1.0f;
            float zlo = (float)(-P.cz), zhi = (float)(P.nz - P.cz);
            if (rz.mz != 0.0f) {
                float t1 = (zlo - rz.za) * rz.inv_mz, t2 = (zhi - rz.za) * rz.inv_mz;
                dlo = fmaxf(dlo, fminf(t1, t2) - 1.0f); dhi = fminf(dhi, fmaxf(t1, t2) + 1.0f);
            } else if (rz.za < zlo || rz.za >= zhi) dhi = dlo - 1.0f;
        }
        float acc = 0.0f;
        int cnt = 0;
        if (dhi > dlo) {
            const int s_lo = max(0, (int)floorf(dlo) + cd), s_hi = min(nd, (int)ceilf(dhi) + cd);
            float d0 = (float)(s_lo - cd);
            float y0 = fmaf(d0, r.m, r.a0), z0 = fmaf(d0, rz.mz, rz.za);
            const size_t kstride = (size_t)nd * nm;
            for (int s = s_lo; s < s_hi; ++s) {
                const float d1 = (float)(s + 1 - cd);
                const float y1 = fmaf(d1, r.m, r.a0), z1 = fmaf(d1, rz.mz, rz.za);
                const float fy0 = floorf(y0), fy1 = floorf(y1), fz0 = floorf(z0), fz1 = floorf(z1);
                float sy = 1.0f, sz = 1.0f;
                if (fy0 != fy1) sy = __saturatef((fmaxf(fy0, fy1) - y0) * r.inv_m);
                if (fz0 != fz1) sz = __saturatef((fmaxf(fz0, fz1) - z0) * rz.inv_mz);
                const float wa = fminf(sy, sz), wb = fmaxf(sy, sz) - wa, wc = 1.0f - fmaxf(sy, sz);
                const int j0 = (int)fy0 + cm, j1 = (int)fy1 + cm, k0 = (int)fz0 + P.cz, k1 = (int)fz1 + P.cz;
                const float *__restrict__ row = base + (size_t)s * nm;
                if (wa > 0.0f && (unsigned)j0 < (unsigned)nm && (unsigned)k0 < (unsigned)P.nz) {
                    if (MODE == 3) ++cnt; else acc = fmaf(wa, __ldg(row + k0 * kstride + j0), acc);
                }
                if (wb > 0.0f) {
                    const int jb = sy < sz ? j1 : j0, kb = sy < sz ? k0 : k1;
                    if ((unsigned)jb < (unsigned)nm && (unsigned)kb < (unsigned)P.nz) {
                        if (MODE == 3) ++cnt; else acc = fmaf(wb, __ldg(row + kb * kstride + jb), acc);
                    }
                }
                if (wc > 0.0f && (unsigned)j1 < (unsigned)nm && (unsigned)k1 < (unsigned)P.nz) {
                    if (MODE == 3) ++cnt; else acc = fmaf(wc, __ldg(row + k1 * kstride + j1), acc);
                }
                y0 = y1; z0 = z1;
            }
        }
        const float Lr = ray_len_L(r, v);
        const float pr = acc * (Lr * r.inv_dd);
        const size_t o = ((size_t)a * P.nv + iv) * P.nu + iu;
        if (MODE == 3) {
            sq = (double)cnt;
        } else if (MODE == 0) {
            out[o] = pr;
        } else if (MODE == 2) {
            out[o] = pr * Lr;          // L * (P f): input of the transpose without a residual
        } else {
            const float T = pr - __ldg(y + o);
            out[o] = T * Lr;           // what the transpose consumes (see back.cu)
            sq = (double)T * (double)T;
        }
    }
    if (MODE == 1 || MODE == 3) {
        double s = block_sum(sq, slot);
        if (threadIdx.x == 0 && threadIdx.y == 0)
            partials[((size_t)blockIdx.z * gridDim.y + blockIdx.y) * gridDim.x + blockIdx.x] = s;
    }
}

cbct_status launch_forward(const cbct_geometry *g, const Level &L, const float *d_vol, const float *d_y,
                           float *d_out, int mode, double *d_sum_sq, cudaStream_t st)
{
    const LevelParams &P = L.p;
    dim3 tb(32, 8), tg((P.nx + 31) / 32, (P.ny + 31) / 32, P.nz);
    if (mode != 3) {
        StageTimer t(g, st, ST_TRANSPOSE);
        transpose_xy_kernel<<<tg, tb, 0, st>>>(d_vol, L.d_volT, P.nx, P.ny);
        CBCT_LAUNCH_CHECK(g);
    }
    dim3 b(FWD_BX, FWD_BY), gr((P.nu + FWD_BX - 1) / FWD_BX, (P.nv + FWD_BY - 1) / FWD_BY, P.np);
    const size_t nblk = (size_t)gr.x * gr.y * gr.z;
    if (mode == 0) {
        StageTimer t(g, st, ST_FORWARD);
        forward_kernel<0><<<gr, b, 0, st>>>(P, d_vol, L.d_volT, L.d_rayu, nullptr, d_out, nullptr);
        CBCT_LAUNCH_CHECK(g);
    } else if (mode == 2) {
        StageTimer t(g, st, ST_FORWARD);
        forward_kernel<2><<<gr, b, 0, st>>>(P, d_vol, L.d_volT, L.d_rayu, nullptr, d_out, nullptr);
        CBCT_LAUNCH_CHECK(g);
    } else {
        if (nblk > (size_t)g->partials_stride) return cbct_fail(CBCT_ERR_INVALID_ARG, "projection stack too large for the reduction buffer");
        {
            StageTimer t(g, st, ST_FORWARD);
            if (mode == 3)
                forward_kernel<3><<<gr, b, 0, st>>>(P, d_vol, L.d_volT, L.d_rayu, nullptr, nullptr, g->d_partials);
            else
                forward_kernel<1><<<gr, b, 0, st>>>(P, d_vol, L.d_volT, L.d_rayu, d_y, d_out, g->d_partials);
            CBCT_LAUNCH_CHECK(g);
        }
        StageTimer t(g, st, ST_REDUCE);
        finalize_sums_kernel<<<1, 256, 0, st>>>(g->d_partials, (int)nblk, 1, g->partials_stride, d_sum_sq);
        CBCT_LAUNCH_CHECK(g);
    }
    return CBCT_OK;
}

extern "C" cbct_status cbct_forward_project(const cbct_geometry *g, int level, const float *d_vol,
                                            float *d_proj, void *cuda_stream)
{
    const Level *L = get_level(g, level);
    if (!L || !d_vol || !d_proj) return cbct_fail(CBCT_ERR_INVALID_ARG, "cbct_forward_project: bad handle, level or NULL buffer");
    return launch_forward(g, *L, d_vol, nullptr, d_proj, 0, nullptr, (cudaStream_t)cuda_stream);
}

extern "C" cbct_status cbct_count_samples(const cbct_geometry *g, int level, unsigned long long *count,
                                          void *cuda_stream)
{
    const Level *L = get_level(g, level);
    if (!L || !count) return cbct_fail(CBCT_ERR_INVALID_ARG, "cbct_count_samples: bad handle, level or NULL");
    cudaStream_t st = (cudaStream_t)cuda_stream;
    cbct_status s = launch_forward(g, *L, nullptr, nullptr, nullptr, 3, g->d_scalars + 10, st);
    if (s != CBCT_OK) return s;
    CBCT_CUDA(cudaMemcpyAsync(g->h_scalars + 10, g->d_scalars + 10, sizeof(double), cudaMemcpyDeviceToHost, st));
    CBCT_CUDA(cudaStreamSynchronize(st));
    *count = (unsigned long long)(g->h_scalars[10] + 0.5);
    return CBCT_OK;
}
