// back.cu -- A3/A4: exact-transpose back-projector, voxel-driven gather.
//
// (P^T T)[voxel] = sum_views sum_rays len(ray ∩ voxel) T[ray] with the SAME len as
// forward.cu ("sum_theta P^T (P f - Y)").  The paper (L187-L191) rejects the
// ray-driven scatter because threads would collide on voxels and evaluates the continuum
// adjoint Eq. 6 instead; here each thread owns voxels and enumerates, per view, every
// detector ray whose slab segment can cross them: the pixel range comes from the voxel ->
// detector map of Eq. A6 (L401-L406) applied to the voxel's extent, and each candidate's
// length is the overlap of three intervals in the slab parameter s in [0,1] -- the same
// fp32 expressions, on the same table entries, as the forward projector's split.
// No atomics, fixed order (views ascending, rows, columns) => deterministic.
//
// Input is T scaled by L(u,v) (ray length source -> pixel), so the per-candidate weight is
// overlap * inv_dd(view, iu).
#include "cbct_internal.cuh"
#include "ray.cuh"
#include "reduce.cuh"

// d_out[ray] = d_in[ray] * L(u,v)
__global__ void scale_by_L_kernel(const LevelParams P, const RayU *__restrict__ rayu,
                                  const float *__restrict__ in, float *__restrict__ out)
{
    const int iu = blockIdx.x * blockDim.x + threadIdx.x;
    const int iv = blockIdx.y, a = blockIdx.z;
    if (iu >= P.nu) return;
    const RayU r = load_rayu(rayu, a * P.nu + iu);
    const float v = fmaf((float)iv, P.dv, P.v0);
    const size_t o = ((size_t)a * P.nv + iv) * P.nu + iu;
    out[o] = __ldg(in + o) * ray_len_L(r, v);
}

constexpr int BK_BX = 32, BK_BY = 4, BK_BZ = 2;

__global__ void __launch_bounds__(BK_BX *BK_BY *BK_BZ)
back_kernel(const LevelParams P, const RayU *__restrict__ rayu, const ViewC *__restrict__ views,
            const float *__restrict__ TL, const float *__restrict__ f, float coef, float *__restrict__ out)
{
    const int i = blockIdx.x * BK_BX + threadIdx.x;
    const int j = blockIdx.y * BK_BY + threadIdx.y;
    const int k = blockIdx.z * BK_BZ + threadIdx.z;
    if (i >= P.nx || j >= P.ny || k >= P.nz) return;
    const float xc = fmaf((float)i, P.hx, P.x0), yc = fmaf((float)j, P.hy, P.y0), zc = fmaf((float)k, P.hz, P.z0);
    const float zlo_mm = zc - 0.5f * P.hz, zhi_mm = zc + 0.5f * P.hz;
    // index-coordinate box of the voxel
    const float bx = (float)(i - P.cx), by = (float)(j - P.cy), bz = (float)(k - P.cz);
    float acc = 0.0f;
    for (int a = 0; a < P.np; ++a) {
        const float4 vw = __ldg(reinterpret_cast<const float4 *>(views) + a);   // c, s, dn, du
        const float rn = fmaf(xc, vw.x, fmaf(yc, vw.y, P.sad));   // (X - S).e_n  > 0
        const float ru = fmaf(xc, vw.y, -yc * vw.x);               // (X - S).e_u
        // bounds of u* = sdd ru/rn and v* = sdd z/rn over the voxel (Eq. A6), conservative
        const float inv_near = P.sdd / (rn - vw.z), inv_far = P.sdd / (rn + vw.z);
        const float ul = ru - vw.w, uh = ru + vw.w;
        const float u_lo = ul * (ul < 0.0f ? inv_near : inv_far), u_hi = uh * (uh > 0.0f ? inv_near : inv_far);
        const float v_lo = zlo_mm * (zlo_mm < 0.0f ? inv_near : inv_far), v_hi = zhi_mm * (zhi_mm > 0.0f ? inv_near : inv_far);
        const int iu_lo = max(0, (int)ceilf((u_lo - P.u0) * P.inv_du - 0.01f));
        const int iu_hi = min(P.nu - 1, (int)floorf((u_hi - P.u0) * P.inv_du + 0.01f));
        const int iv_lo = max(0, (int)ceilf((v_lo - P.v0) * P.inv_dv - 0.01f));
        const int iv_hi = min(P.nv - 1, (int)floorf((v_hi - P.v0) * P.inv_dv + 0.01f));
        if (iu_lo > iu_hi || iv_lo > iv_hi) continue;
        const float *__restrict__ Ta = TL + (size_t)a * P.nv * P.nu;
        for (int iu = iu_lo; iu <= iu_hi; ++iu) {
            const RayU r = load_rayu(rayu, a * P.nu + iu);
            const float d0 = r.drive ? by : bx, mn = r.drive ? bx : by;   // slab coordinate, minor plane
            // in-plane: s-interval where minor(s) = y0 + s m lies in [mn, mn+1)
            const float y0 = fmaf(d0, r.m, r.a0);
            const float t1 = (mn - y0) * r.inv_m, t2 = (mn + 1.0f - y0) * r.inv_m;
            const float s_lo = fmaxf(fminf(t1, t2), 0.0f), s_hi = fminf(fmaxf(t1, t2), 1.0f);
            if (!(s_hi > s_lo)) continue;
            float col = 0.0f;
            for (int iv = iv_lo; iv <= iv_hi; ++iv) {
                const float v = fmaf((float)iv, P.dv, P.v0);
                const RayZ rz = ray_z(r, v, P.sz);
                const float z0 = fmaf(d0, rz.mz, rz.za);
                const float q1 = (bz - z0) * rz.inv_mz, q2 = (bz + 1.0f - z0) * rz.inv_mz;
                const float lo = fmaxf(fminf(q1, q2), s_lo), hi = fminf(fmaxf(q1, q2), s_hi);
                const float w = hi - lo;
                if (w > 0.0f) col = fmaf(w, __ldg(Ta + (size_t)iv * P.nu + iu), col);
            }
            acc = fmaf(col, r.inv_dd, acc);
        }
    }
    const size_t o = ((size_t)k * P.ny + j) * P.nx + i;
    out[o] = f ? fmaf(-coef, acc, __ldg(f + o)) : acc;
}

cbct_status launch_back(const cbct_geometry *g, const Level &L, const float *d_in, int scaled,
                        const float *d_f, float coef, float *d_out, cudaStream_t st)
{
    const LevelParams &P = L.p;
    const float *src = d_in;
    if (!scaled) {
        StageTimer t(g, st, ST_TRANSFER);
        dim3 b(128), gr((P.nu + 127) / 128, P.nv, P.np);
        scale_by_L_kernel<<<gr, b, 0, st>>>(P, L.d_rayu, d_in, L.d_T);
        CBCT_LAUNCH_CHECK(g);
        src = L.d_T;
    }
    dim3 b(BK_BX, BK_BY, BK_BZ);
    dim3 gr((P.nx + BK_BX - 1) / BK_BX, (P.ny + BK_BY - 1) / BK_BY, (P.nz + BK_BZ - 1) / BK_BZ);
    StageTimer t(g, st, ST_BACK);
    back_kernel<<<gr, b, 0, st>>>(P, L.d_rayu, L.d_view, src, d_f, coef, d_out);
    CBCT_LAUNCH_CHECK(g);
    return CBCT_OK;
}

extern "C" cbct_status cbct_back_project(const cbct_geometry *g, int level, const float *d_proj,
                                         float *d_vol, void *cuda_stream)
{
    const Level *L = get_level(g, level);
    if (!L || !d_proj || !d_vol) return cbct_fail(CBCT_ERR_INVALID_ARG, "cbct_back_project: bad handle, level or NULL buffer");
    return launch_back(g, *L, d_proj, 0, nullptr, 0.0f, d_vol, (cudaStream_t)cuda_stream);
}
