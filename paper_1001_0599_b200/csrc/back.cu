// back.cu -- A3/A4: exact-transpose back-projector, voxel-driven gather.
//
// (P^T T)[voxel] = sum_views sum_rays len(ray ∩ voxel) T[ray] with the SAME len as
// forward.cu ("sum_theta P^T (P f - Y)").  The paper (L187-L191) rejects the
// ray-driven scatter because threads would collide on voxels and evaluates the continuum
// adjoint Eq. 6 instead; here each thread owns voxels and enumerates, per view, every
// detector ray whose slab segment can cross them: the pixel range comes from the voxel ->
// detector map of Eq. A6 (L401-L406) applied to the voxel's extent (to first order, with
// inflated half extents, so one reciprocal serves both detector axes), and each candidate's
// length is the overlap of three intervals in the slab parameter t in [0,1] -- the same
// fp32 crossing parameters, from the same table entries, as the forward projector's
// (ray.cuh).  No atomics, fixed order (views ascending, columns, rows) => deterministic.
//
// Input is T scaled by L(u,v) (ray length source -> pixel), so the per-candidate weight is
// overlap * inv_dd(view, iu).
//
// Rotation symmetry (R == 4, see forward.cu): a thread owns the four quarter-turn images
// w_0..w_3 of a voxel of the first quadrant.  For a base view t and the image w_s, the
// weights a(ray(t; iu, iv), w_s) are also those of the pairs (view t + 90 r, voxel w_{s+r}),
// so each weight is computed once and applied to four accumulators with ONE 16-byte load
// from the interleaved residual stack T4[base view][iu][iv][r] (detector rows fastest, matching the lanes).
//
// Mirror symmetry (M == 2): with the volume centred in z and the detector in v, the weight of
// (ray (iu, iv), voxel k) is also that of (ray (iu, nv-1-iv), voxel nz-1-k): the thread owns
// both voxels and adds a second load per weight.
#include "cbct_internal.cuh"
#include "ray.cuh"
#include "reduce.cuh"

// d_out = d_in * L(u,v) in the d_T layout (plain for R == 1, quarter-turn interleaved for R == 4)
template <int R>
__global__ void scale_by_L_kernel(const LevelParams P, const RayU *__restrict__ rayu,
                                  const float *__restrict__ in, float *__restrict__ out)
{
    const int iu = blockIdx.x * blockDim.x + threadIdx.x;
    const int iv = blockIdx.y, a = blockIdx.z;
    if (iu >= P.nu) return;
    const RayU r = load_rayu(rayu, a * P.nu + iu);
    const float v = fmaf((float)iv, P.dv, P.v0);
    const float Lr = ray_len_L(r, v);
    const size_t plane = (size_t)P.nv * P.nu, pix = (size_t)iv * P.nu + iu;
    float res[R];
#pragma unroll
    for (int q = 0; q < R; ++q) res[q] = __ldg(in + (size_t)(a + q * P.nbase) * plane + pix) * Lr;
    const size_t ot = ((size_t)a * P.nu + iu) * P.nv + iv;          // d_T layout: detector rows fastest
    if (R == 4) reinterpret_cast<float4 *>(out)[ot] = make_float4(res[0], res[1 % R], res[2 % R], res[3 % R]);
    else out[ot] = res[0];
}

constexpr int BK_BZ = 32, BK_BX = 8;       // block: 32 consecutive k (lanes) x 8 consecutive i

template <int R, int M>
__global__ void __launch_bounds__(BK_BZ *BK_BX)
back_kernel(const LevelParams P, const RayU *__restrict__ rayu, const ViewC *__restrict__ views,
            const float *__restrict__ TL, const float *__restrict__ f, float coef, float *__restrict__ out)
{
    // lanes run along z: a warp shares (i,j), hence the whole in-plane part of every candidate test
    // (uniform branches, broadcast table loads), and its lanes read consecutive detector rows
    const int k = blockIdx.z * BK_BZ + threadIdx.x;
    const int i = blockIdx.x * BK_BX + threadIdx.y;
    const int j = blockIdx.y;
    const int ni = R == 4 ? P.nx / 2 : P.nx;
    if (i >= ni || k >= P.nz / M) return;           // M == 2: the upper half are the mirror images nz-1-k
    const float zc = fmaf((float)k, P.hz, P.z0);
    const float zlo_mm = zc - 0.5f * P.hz, zhi_mm = zc + 0.5f * P.hz;
    const float bz = (float)(k - P.cz), bz1 = bz + 1.0f;
    // the R quarter-turn images of the voxel: (i,j), (n-1-j, i), (n-1-i, n-1-j), (j, n-1-i)
    int vi[R], vj[R];
    vi[0] = i; vj[0] = j;
    if (R == 4) {
        const int n1 = P.nx - 1;
        vi[1 % R] = n1 - j; vj[1 % R] = i;
        vi[2 % R] = n1 - i; vj[2 % R] = n1 - j;
        vi[3 % R] = j;      vj[3 % R] = n1 - i;
    }
    float acc[R * M];
#pragma unroll
    for (int q = 0; q < R * M; ++q) acc[q] = 0.0f;
    const size_t plane = (size_t)P.nv * P.nu;
    for (int a = 0; a < P.nbase; ++a) {
        const float4 vw = __ldg(reinterpret_cast<const float4 *>(views) + a);   // c, s, dn, du
        const float *__restrict__ Ta = TL + (size_t)a * plane * R;
#pragma unroll
        for (int sg = 0; sg < R; ++sg) {
            const float xc = fmaf((float)vi[sg], P.hx, P.x0), yc = fmaf((float)vj[sg], P.hy, P.y0);
            const float bx = (float)(vi[sg] - P.cx), by = (float)(vj[sg] - P.cy);
            const float rn = fmaf(xc, vw.x, fmaf(yc, vw.y, P.sad));   // (X - S).e_n  > 0
            const float ru = fmaf(xc, vw.y, -yc * vw.x);               // (X - S).e_u
            // shadow of the voxel on the detector (Eq. A6): u* = sdd ru/rn, v* = sdd z/rn, to first
            // order in the voxel's half extents dn, du (inflated in the table), plus 0.02 pixel
            float rinv;
            asm("rcp.approx.ftz.f32 %0, %1;" : "=f"(rinv) : "f"(rn));
            const float mag = P.sdd * rinv, tn = ru * rinv, e = vw.z * rinv;
            const float uc = mag * ru, W = mag * fmaf(fabsf(tn), vw.z, vw.w);
            const float v_lo = zlo_mm * mag * (zlo_mm < 0.0f ? 1.0f + e : 1.0f - e);
            const float v_hi = zhi_mm * mag * (zhi_mm > 0.0f ? 1.0f + e : 1.0f - e);
            const int iu_lo = max(0, __float2int_ru((uc - W - P.u0) * P.inv_du - 0.02f));
            const int iu_hi = min(P.nu - 1, __float2int_rd((uc + W - P.u0) * P.inv_du + 0.02f));
            const int iv_lo = max(0, __float2int_ru((v_lo - P.v0) * P.inv_dv - 0.02f));
            const int iv_hi = min(P.nv - 1, __float2int_rd((v_hi - P.v0) * P.inv_dv + 0.02f));
            if (iv_lo > iv_hi) continue;
            for (int iu = iu_lo; iu <= iu_hi; ++iu) {
                const RayU r = load_rayu(rayu, a * P.nu + iu);
                const float d0 = r.drive ? by : bx, mn = r.drive ? bx : by;   // slab coordinate, minor plane
                // in-plane: t-interval where minor(t) = y0 + t m lies in [mn, mn+1)
                const float y0 = fmaf(d0, r.m, r.a0);
                const float t1 = (mn - y0) * r.inv_m, t2 = (mn + 1.0f - y0) * r.inv_m;
                const float s_lo = fmaxf(fminf(t1, t2), 0.0f), s_hi = fminf(fmaxf(t1, t2), 1.0f);
                if (!(s_hi > s_lo)) continue;
                float col[R * M];
#pragma unroll
                for (int q = 0; q < R * M; ++q) col[q] = 0.0f;
                for (int iv = iv_lo; iv <= iv_hi; ++iv) {
                    const float v = fmaf((float)iv, P.dv, P.v0);
                    const RayZ rz = ray_z(r, v, P.sz);
                    const float z0 = fmaf(d0, rz.mz, rz.za);
                    const float q1 = (bz - z0) * rz.inv_mz, q2 = (bz1 - z0) * rz.inv_mz;
                    const float lo = fmaxf(fminf(q1, q2), s_lo), hi = fminf(fmaxf(q1, q2), s_hi);
                    const float w = hi - lo;
                    if (w > 0.0f) {
#pragma unroll
                        for (int mm = 0; mm < M; ++mm) {        // the mirror voxel sees the mirror row with the same weight
                            const size_t ot = (size_t)iu * P.nv + (mm ? P.nv - 1 - iv : iv);
                            if (R == 4) {
                                const float4 t = __ldg(reinterpret_cast<const float4 *>(Ta) + ot);
                                col[mm * R] = fmaf(w, t.x, col[mm * R]);
                                col[mm * R + 1 % R] = fmaf(w, t.y, col[mm * R + 1 % R]);
                                col[mm * R + 2 % R] = fmaf(w, t.z, col[mm * R + 2 % R]);
                                col[mm * R + 3 % R] = fmaf(w, t.w, col[mm * R + 3 % R]);
                            } else {
                                col[mm * R] = fmaf(w, __ldg(Ta + ot), col[mm * R]);
                            }
                        }
                    }
                }
                // weights of image sg under base view a serve the pairs (view a + r nbase, image sg + r)
#pragma unroll
                for (int mm = 0; mm < M; ++mm)
#pragma unroll
                    for (int q = 0; q < R; ++q)
                        acc[mm * R + (sg + q) % R] = fmaf(col[mm * R + q], r.inv_dd, acc[mm * R + (sg + q) % R]);
            }
        }
    }
#pragma unroll
    for (int mm = 0; mm < M; ++mm)
#pragma unroll
        for (int q = 0; q < R; ++q) {
            const size_t o = ((size_t)(mm ? P.nz - 1 - k : k) * P.ny + vj[q]) * P.nx + vi[q];
            out[o] = f ? fmaf(-coef, acc[mm * R + q], __ldg(f + o)) : acc[mm * R + q];
        }
}

cbct_status launch_back(const cbct_geometry *g, const Level &L, const float *d_in, int scaled,
                        const float *d_f, float coef, float *d_out, cudaStream_t st)
{
    const LevelParams &P = L.p;
    const float *src = d_in;
    if (!scaled) {
        StageTimer t(g, st, ST_TRANSFER);
        dim3 b(128), gr((P.nu + 127) / 128, P.nv, P.nbase);
        if (P.nsym == 4) scale_by_L_kernel<4><<<gr, b, 0, st>>>(P, L.d_rayu, d_in, L.d_T);
        else scale_by_L_kernel<1><<<gr, b, 0, st>>>(P, L.d_rayu, d_in, L.d_T);
        CBCT_LAUNCH_CHECK(g);
        src = L.d_T;
    }
    StageTimer t(g, st, ST_BACK);
    dim3 b(BK_BZ, BK_BX);
    const int nzh = P.nz / P.nmir;
    if (P.nsym == 4) {
        dim3 gr((P.nx / 2 + BK_BX - 1) / BK_BX, P.ny / 2, (nzh + BK_BZ - 1) / BK_BZ);
        if (P.nmir == 2) back_kernel<4, 2><<<gr, b, 0, st>>>(P, L.d_rayu, L.d_view, src, d_f, coef, d_out);
        else back_kernel<4, 1><<<gr, b, 0, st>>>(P, L.d_rayu, L.d_view, src, d_f, coef, d_out);
    } else {
        dim3 gr((P.nx + BK_BX - 1) / BK_BX, P.ny, (nzh + BK_BZ - 1) / BK_BZ);
        if (P.nmir == 2) back_kernel<1, 2><<<gr, b, 0, st>>>(P, L.d_rayu, L.d_view, src, d_f, coef, d_out);
        else back_kernel<1, 1><<<gr, b, 0, st>>>(P, L.d_rayu, L.d_view, src, d_f, coef, d_out);
    }
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
