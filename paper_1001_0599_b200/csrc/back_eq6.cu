// back_eq6.cu -- NEXT-1 of the scope table: the paper's OWN gradient of the data term, Eq. (6)
// (PAPER.md:L195-L199), next to the exact transpose of back.cu.
//
//     b6(X) = (dV / (du dv)) * sum_theta  L^3(u*,v*) / (L0 l^2(X)) * T^theta(u*, v*)
//
// (u*, v*) is where the line source -> voxel centre X meets the imager (Eq. A6), l = |X - S|,
// L = sqrt(L0^2 + u*^2 + v*^2) (A2, L374), the prefactor is the Jacobian of Eq. A7 (L412) and T^theta(u*,v*) is
// taken by bilinear interpolation between pixel centres (L199).  The factor dV/(du dv) puts b6 on the scale
// of P^T T (reading S1), so it can stand in for it in step 1 of Algorithm A1 -- an UNMATCHED
// projector pair, which is what the paper ran.  A tap outside the detector is 0 (reading S19).
//
// Since l = L rn / L0 with rn = (X - S).e_n, the prefactor is  L^3/(L0 l^2) = L L0 / rn^2:  one square root per
// voxel and view.  One thread owns EQ6_KZ consecutive voxels of a z-column, lanes run along x: per view the
// in-plane part (rn, u*, the two u-taps and their weights) is computed once per column, the lanes' taps are
// neighbours on a detector row (coalesced gathers from the plain [view][row][column] stack), and the volume is
// written with coalesced stores.  Hardware texture filtering is not used: its 8-bit weights cannot meet the
// 1e-5 tolerance.  No atomics, fixed summation order (views ascending).
#include "cbct_internal.cuh"

constexpr int EQ6_KZ = 8, EQ6_BX = 32, EQ6_BY = 4;

// The detector coordinates (u*, v*) decide interpolation weights between pixels whose values may differ by
// O(1): at 512 pixels across, fp32 coordinates (ulp 6e-5 pixel) alone would cost ~1e-5 of the result.  The
// coordinate chain of a z-column and view therefore runs in fp64, once for the EQ6_KZ voxels of a thread; the
// voxels' row offsets from the first, the weights, samples and sums are fp32.
struct Eq6Params {
    double x0, y0, z0, hx, hy, hz;     // centre of voxel 0, voxel size (mm)
    double u0, v0, inv_du, inv_dv;     // centre of pixel 0, 1 / pitch
    double sad, sdd;
};

__global__ void __launch_bounds__(EQ6_BX *EQ6_BY)
back_eq6_kernel(const LevelParams P, const Eq6Params E, const double2 *__restrict__ cs, const float *__restrict__ T,
                const float *__restrict__ f, float coef, float scale, float *__restrict__ out)
{
    const int i = blockIdx.x * EQ6_BX + threadIdx.x;
    const int j = blockIdx.y * EQ6_BY + threadIdx.y;
    const int k0 = blockIdx.z * EQ6_KZ;
    if (i >= P.nx || j >= P.ny) return;
    const double xc = fma((double)i, E.hx, E.x0), yc = fma((double)j, E.hy, E.y0);
    const double z_first = fma((double)k0, E.hz, E.z0);
    float acc[EQ6_KZ];
#pragma unroll
    for (int t = 0; t < EQ6_KZ; ++t) acc[t] = 0.0f;
    const float sdd2 = (float)(E.sdd * E.sdd);
    const size_t plane = (size_t)P.nv * P.nu;
    for (int a = 0; a < P.np; ++a) {
        const double2 c = __ldg(cs + a);                                         // cos, sin of the view angle
        const double rn = fma(xc, c.x, fma(yc, c.y, E.sad));                     // (X - S).e_n > 0
        const double ru = fma(xc, c.y, -yc * c.x);                               // (X - S).e_u
        const double rinv = 1.0 / rn;
        const double mag = E.sdd * rinv;
        const double us = mag * ru;
        const float pre = (float)(E.sdd * rinv * rinv);                          // L0 / rn^2
        // the two detector columns around u* and, per voxel, the two rows around v*; v* = mag * z is linear in k: the
        // row coordinate of the thread's first voxel is split in fp64 into an integer and a fraction; the thread's other
        // voxels are at most EQ6_KZ * (rows per voxel) further, where fp32 still resolves 1e-6 of a row
        const double fu = (us - E.u0) * E.inv_du;
        const double fu0 = floor(fu);
        const float tu = (float)(fu - fu0);
        const int iu0 = (int)fu0;
        const float *__restrict__ Ta = T + (size_t)a * plane;
        const float usf = (float)us;
        const float lu2 = fmaf(usf, usf, sdd2);
        const double fv_first = (mag * z_first - E.v0) * E.inv_dv;
        const double fv_base = floor(fv_first);
        const int iv_base = (int)fv_base;
        const float rv_first = (float)(fv_first - fv_base), dfv = (float)(mag * E.hz * E.inv_dv);
        const float vs_first = (float)(mag * z_first), dvs = (float)(mag * E.hz);
        // rows the thread's voxels can touch: iv_base + floor(rv_first + t dfv) + {0,1}, t = 0 .. EQ6_KZ-1
        const int iv_a = iv_base + (int)floorf(fminf(rv_first, fmaf((float)(EQ6_KZ - 1), dfv, rv_first)));
        const int iv_b = iv_base + (int)floorf(fmaxf(rv_first, fmaf((float)(EQ6_KZ - 1), dfv, rv_first))) + 1;
        auto prefactor = [&](int t) {           // L0 L / rn^2 with L = sqrt(L0^2 + u*^2 + v*^2)
            const float vs = fmaf((float)t, dvs, vs_first);
            float Lr;
            asm("sqrt.approx.ftz.f32 %0, %1;" : "=f"(Lr) : "f"(fmaf(vs, vs, lu2)));
            return pre * Lr;
        };
        if (iu0 >= 0 && iu0 + 1 < P.nu && iv_a >= 0 && iv_b < P.nv) {
            // every tap of every voxel of the thread is on the detector: no tests, one address per row pair
            const float *__restrict__ Tc = Ta + iu0;
#pragma unroll
            for (int t = 0; t < EQ6_KZ; ++t) {
                const float xv = fmaf((float)t, dfv, rv_first);
                const float xv0 = floorf(xv), tv = xv - xv0;
                const float *__restrict__ r0 = Tc + (iv_base + (int)xv0) * P.nu;
                const float *__restrict__ r1 = r0 + P.nu;
                const float t00 = __ldg(r0), t01 = __ldg(r0 + 1), t10 = __ldg(r1), t11 = __ldg(r1 + 1);
                const float lo = fmaf(tu, t01 - t00, t00), hi = fmaf(tu, t11 - t10, t10);
                acc[t] = fmaf(prefactor(t), fmaf(tv, hi - lo, lo), acc[t]);
            }
        } else if (iu0 + 1 >= 0 && iu0 < P.nu && iv_b >= 0 && iv_a < P.nv) {
            // near the detector's edge: a tap outside the detector is 0
            const float wu0 = (iu0 >= 0 && iu0 < P.nu) ? 1.0f - tu : 0.0f;
            const float wu1 = (iu0 + 1 >= 0 && iu0 + 1 < P.nu) ? tu : 0.0f;
            const int c0 = min(max(iu0, 0), P.nu - 1), c1 = min(max(iu0 + 1, 0), P.nu - 1);
#pragma unroll
            for (int t = 0; t < EQ6_KZ; ++t) {
                const float xv = fmaf((float)t, dfv, rv_first);
                const float xv0 = floorf(xv), tv = xv - xv0;
                const int iv0 = iv_base + (int)xv0;
                const float wv0 = (iv0 >= 0 && iv0 < P.nv) ? 1.0f - tv : 0.0f;
                const float wv1 = (iv0 + 1 >= 0 && iv0 + 1 < P.nv) ? tv : 0.0f;
                const int r0 = min(max(iv0, 0), P.nv - 1) * P.nu, r1 = min(max(iv0 + 1, 0), P.nv - 1) * P.nu;
                const float t00 = __ldg(Ta + r0 + c0), t01 = __ldg(Ta + r0 + c1);
                const float t10 = __ldg(Ta + r1 + c0), t11 = __ldg(Ta + r1 + c1);
                const float val = wv0 * fmaf(wu1, t01, wu0 * t00) + wv1 * fmaf(wu1, t11, wu0 * t10);
                acc[t] = fmaf(prefactor(t), val, acc[t]);
            }
        }
    }
#pragma unroll
    for (int t = 0; t < EQ6_KZ; ++t) {
        const int k = k0 + t;
        if (k < P.nz) {
            const size_t o = ((size_t)k * P.ny + j) * P.nx + i;
            const float v = scale * acc[t];
            out[o] = f ? fmaf(-coef, v, __ldg(f + o)) : v;
        }
    }
}

// out = f - coef * b6(T) (f may be NULL: out = b6(T)); T in the plain [view][row][column] layout
cbct_status launch_back_eq6(const cbct_geometry *g, const Level &L, const float *d_T, const float *d_f, float coef,
                            float *d_out, cudaStream_t st)
{
    const LevelParams &P = L.p;
    StageTimer t(g, st, ST_BACK);
    dim3 b(EQ6_BX, EQ6_BY), gr((P.nx + EQ6_BX - 1) / EQ6_BX, (P.ny + EQ6_BY - 1) / EQ6_BY, (P.nz + EQ6_KZ - 1) / EQ6_KZ);
    const float scale = (float)(L.hx * L.hy * L.hz / (L.du * L.dv));
    const cbct_geometry_desc &d = g->desc;
    Eq6Params E;
    E.hx = L.hx; E.hy = L.hy; E.hz = L.hz;
    E.x0 = -0.5 * (P.nx - 1) * L.hx + d.vol_off[0];
    E.y0 = -0.5 * (P.ny - 1) * L.hy + d.vol_off[1];
    E.z0 = -0.5 * (P.nz - 1) * L.hz + d.vol_off[2];
    E.u0 = -0.5 * (P.nu - 1) * L.du + d.det_off_u;
    E.v0 = -0.5 * (P.nv - 1) * L.dv + d.det_off_v;
    E.inv_du = 1.0 / L.du; E.inv_dv = 1.0 / L.dv;
    E.sad = d.sad; E.sdd = d.sdd;
    back_eq6_kernel<<<gr, b, 0, st>>>(P, E, L.d_cs, d_T, d_f, coef, scale, d_out);
    CBCT_LAUNCH_CHECK(g);
    return CBCT_OK;
}

extern "C" cbct_status cbct_back_project_eq6(const cbct_geometry *g, int level, const float *d_proj,
                                             float *d_vol, void *cuda_stream)
{
    const Level *L = get_level(g, level);
    if (!L || !d_proj || !d_vol) return cbct_fail(CBCT_ERR_INVALID_ARG, "cbct_back_project_eq6: bad handle, level or NULL buffer");
    return launch_back_eq6(g, *L, d_proj, nullptr, 0.0f, d_vol, (cudaStream_t)cuda_stream);
}
