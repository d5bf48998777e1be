// ray.cuh -- the ray parametrisation shared by the forward projector and its transpose.
// Both kernels evaluate these few fp32 expressions on the same table entries, so the
// coefficient a(ray, voxel) they compute is the same number on both sides (PAPER.md:L91
// Eq. 1 for the ray, L187 for P and P^T sharing one matrix).
//
// Along the driving coordinate D (index units, slab s spans D in [s - cd, s + 1 - cd]):
//     minor(D) = a0 + D m                       |m| <= 1
//     z(D)     = za + D mz,   mz = v q,  za = sz - sd mz        |mz| <= 1 (checked at create)
// Inside the slab starting at D0 the ray is written  y(t) = y0 + t m,  z(t) = z0 + t mz,
// t in [0,1], with y0 = fma(D0, m, a0), z0 = fma(D0, mz, za); it crosses the grid plane
// `c` of the minor axis at t = (c - y0) inv_m and of z at t = (c - z0) inv_mz.  Every weight
// of either projector is a difference of such crossing parameters clipped to [0,1].
#pragma once
#include "cbct_internal.cuh"

struct RayZ {
    float mz, za, inv_mz;
};

// 1 / (x + tiny): finite for x == 0 (a ray lying in a z-plane never crosses one), a single
// MUFU.RCP otherwise.  The approximation is a deterministic function of x, and both
// projectors call it on the same x.
__device__ __forceinline__ float ray_rcp(float x)
{
    float r;
    asm("rcp.approx.ftz.f32 %0, %1;" : "=f"(r) : "f"(x + 1.0e-37f));
    return r;
}

__device__ __forceinline__ RayZ ray_z(const RayU &r, float v, float sz)
{
    RayZ z;
    z.mz = v * r.q;
    z.za = fmaf(-r.sd, z.mz, sz);
    z.inv_mz = ray_rcp(z.mz);
    return z;
}

// length in mm of the whole ray source -> pixel; one unit slab holds L * inv_dd of it
__device__ __forceinline__ float ray_len_L(const RayU &r, float v) { return sqrtf(fmaf(v, v, r.c_l)); }

// Position of detector row iv inside its column of the residual stack: plain, or split by row parity (LevelParams::tP,
// back_tma.cu).  The stack holds L(u,v) * inv_dd(view, iu) * T: the length of one unit slab of the ray times the residual,
// so that a back-projector's weight is the bare overlap of crossing parameters.
__device__ __forceinline__ int t_row_slot(const LevelParams &P, int iv)
{
    return P.tP == 2 ? (iv & 1) * P.tXP + (iv >> 1) : iv;
}

__device__ __forceinline__ RayU load_rayu(const RayU *__restrict__ t, int idx)
{
    const float4 *p = reinterpret_cast<const float4 *>(t + idx);
    float4 A = __ldg(p), B = __ldg(p + 1);
    RayU r;
    r.a0 = A.x; r.m = A.y; r.inv_m = A.z; r.q = A.w;
    r.sd = B.x; r.inv_dd = B.y; r.c_l = B.z; r.drive = __float_as_int(B.w);
    return r;
}
