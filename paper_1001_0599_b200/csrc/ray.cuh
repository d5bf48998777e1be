// ray.cuh -- the ray parametrisation shared by the forward projector and its transpose.
// Both kernels evaluate these few fp32 expressions on the same table entries, so the
// coefficient a(ray, voxel) they compute is the same number on both sides.
#pragma once
#include "cbct_internal.cuh"

struct RayZ {
    float mz, za, inv_mz;   // z(D) = za + D * mz  in index coordinates
};

__device__ __forceinline__ RayZ ray_z(const RayU &r, float v, float sz)
{
    RayZ z;
    z.mz = v * r.q;
    z.za = fmaf(-r.sd, z.mz, sz);
    z.inv_mz = (z.mz == 0.0f) ? 1.0e30f : __frcp_rn(z.mz);
    return z;
}

// length in mm of the ray inside one unit slab of its driving axis
__device__ __forceinline__ float ray_len_L(const RayU &r, float v) { return sqrtf(fmaf(v, v, r.c_l)); }

__device__ __forceinline__ RayU load_rayu(const RayU *__restrict__ t, int idx)
{
    const float4 *p = reinterpret_cast<const float4 *>(t + idx);
    float4 A = __ldg(p), B = __ldg(p + 1);
    RayU r;
    r.a0 = A.x; r.m = A.y; r.inv_m = A.z; r.q = A.w;
    r.sd = B.x; r.inv_dd = B.y; r.c_l = B.z; r.drive = __float_as_int(B.w);
    return r;
}
