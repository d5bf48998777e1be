// back.cu -- A3/A4: exact-transpose back-projector, voxel-driven gather.
//
// (P^T T)[voxel] = sum_views sum_rays len(ray ∩ voxel) T[ray] with the SAME len as
// forward.cu ("sum_theta P^T (P f - Y)").  The paper (L187-L191) rejects the
// ray-driven scatter because threads would collide on voxels and evaluates the continuum
// adjoint Eq. 6 instead; here each thread owns voxels and enumerates, per view, every
// detector ray whose slab segment crosses them: the column range comes from the voxel ->
// detector map of Eq. A6 (L401-L406) applied to the voxel's in-plane extent (to first order,
// with inflated half extents), the row range per column is exact (see back_kernel), and each
// ray's length is the overlap of three intervals in the slab parameter t in [0,1] -- the same
// fp32 crossing parameters, from the same table entries, as the forward projector's
// (ray.cuh).  No atomics, fixed order (views ascending, columns, rows) => deterministic.
//
// Input is T scaled by L(u,v) inv_dd(view, iu) (the length of one unit slab of the ray), so the per-candidate weight
// is the bare overlap.
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

// d_out = d_in * L(u,v) * inv_dd(view, iu) in the d_T layout (plain for R == 1, quarter-turn interleaved for R == 4)
template <int R>
__global__ void scale_by_L_kernel(const LevelParams P, const RayU *__restrict__ rayu,
                                  const float *__restrict__ in, float *__restrict__ out)
{
    const int iu = blockIdx.x * blockDim.x + threadIdx.x;
    const int iv = blockIdx.y, a = blockIdx.z;
    if (iu >= P.nu) return;
    const RayU r = load_rayu(rayu, a * P.nu + iu);
    const float v = fmaf((float)iv, P.dv, P.v0);
    const float Lr = ray_len_L(r, v) * r.inv_dd;
    const size_t plane = (size_t)P.nv * P.nu, pix = (size_t)iv * P.nu + iu;
    float res[R];
#pragma unroll
    for (int q = 0; q < R; ++q) res[q] = __ldg(in + (size_t)(a + q * P.nbase) * plane + pix) * Lr;
    const size_t ot = ((size_t)a * P.nu + iu) * P.nv + t_row_slot(P, iv);   // d_T layout: detector rows fastest
    if (R == 4) reinterpret_cast<float4 *>(out)[ot] = make_float4(res[0], res[1 % R], res[2 % R], res[3 % R]);
    else out[ot] = res[0];
}

constexpr int BK_BX = 8;       // block: one warp (lanes along z) per i, 8 consecutive i

// Lanes run along z, so a warp shares (i,j) and with it the whole in-plane part of every candidate
// (uniform branches, broadcast table loads); each thread owns KT voxels k = k0 + lane + 32 t of the column,
// which spreads that in-plane part over KT times as many voxels (KT = 2 with 80 registers measured best at 256^3:
// the kernel is bound by load latency, so occupancy is worth more than a longer amortisation).
//
// Per (base view, voxel image, detector column iu) the in-plane part gives the slab interval
// [s_lo, s_hi] of t in which the ray is above the voxel's (i,j) square.  There the ray climbs
// from z = sz + v cA to sz + v cB, c = q (D - sd) > 0, so the rows v that can reach a voxel
// [zl, zh] + sz are  v in ( zl / c_far , zh / c_near )  (with the roles of c_near / c_far set by the
// signs of zl, zh): an exact row range from two reciprocals per column, and every row in it is a hit.
// The row's weight is the overlap of [s_lo, s_hi] with the t-interval between its crossings of the
// voxel's two z-planes, t = z_plane / (v q) - (d0 - sd): the same crossing parameters as
// forward.cu's, written relative to the source so that one reciprocal serves both planes.
// One detector column's contribution to the KT voxels of a thread.  In: the slab interval [s_lo, s_hi] of the column's ray
// above the voxel's (i,j) square, e = slab start relative to the source, q, inv_dd of the ray, 1/c at the two ends of
// the interval, and the 32-bit entry offset oA of the column's row 0 in the residual stack T (float4 entries for
// R == 4, floats for R == 1).  SG = the voxel image the interval belongs to: its weights serve the pairs
// (view a + r nbase, image SG + r); the mirror voxel sees the mirror row nv-1-iv with the same weight.
template <int R, int M, int KT, int SG>
__device__ __forceinline__ void gather_column(float (&acc)[KT][R * M], const float (&zl)[KT], const LevelParams &P,
                                              const float *__restrict__ T, float c0v, float s_lo, float s_hi, float e,
                                              float q, float inv_dd, float ic_near, float ic_far, int oA)
{
    const float tiny = copysignf(1.0e-37f, q);            // a row with v == 0 counts as v = 0+
    const int oB = oA + P.nv - 1;                         // row nv-1
#pragma unroll
    for (int t = 0; t < KT; ++t) {
        const float zlo = zl[t], zhi = zlo + 1.0f;
        const float v_lo = zlo * (zlo >= 0.0f ? ic_far : ic_near);
        const float v_hi = zhi * (zhi >= 0.0f ? ic_near : ic_far);
        int iv = max(0, __float2int_ru(fmaf(v_lo, P.inv_dv, c0v) - 2.0e-3f));
        const int iv_hi = min(P.nv - 1, __float2int_rd(fmaf(v_hi, P.inv_dv, c0v) + 2.0e-3f));
        if (iv > iv_hi) continue;
        // overlap of [s_lo, s_hi] with the t-interval between the row's crossings of the voxel's z-planes,
        // times the slab length per unit of L (inv_dd); rows of the exact range always overlap
        auto weight = [&](int row) {
            const float v = fmaf((float)row, P.dv, P.v0);
            float inv;
            asm("rcp.approx.ftz.f32 %0, %1;" : "=f"(inv) : "f"(fmaf(v, q, tiny)));
            const float q1 = fmaf(zlo, inv, -e), q2 = fmaf(zhi, inv, -e);
            const float lo = fmaxf(fminf(q1, q2), s_lo), hi = fminf(fmaxf(q1, q2), s_hi);
            return fmaxf(hi - lo, 0.0f);          // the slab length per unit of L (inv_dd) is folded into T
        };
        auto gather = [&](float w, const float4 &tA, const float4 &tB) {
            acc[t][(SG + 0) % R] = fmaf(w, tA.x, acc[t][(SG + 0) % R]);
            if (R == 4) {
                acc[t][(SG + 1) % R] = fmaf(w, tA.y, acc[t][(SG + 1) % R]);
                acc[t][(SG + 2) % R] = fmaf(w, tA.z, acc[t][(SG + 2) % R]);
                acc[t][(SG + 3) % R] = fmaf(w, tA.w, acc[t][(SG + 3) % R]);
            }
            if (M == 2) {
                acc[t][R + (SG + 0) % R] = fmaf(w, tB.x, acc[t][R + (SG + 0) % R]);
                if (R == 4) {
                    acc[t][R + (SG + 1) % R] = fmaf(w, tB.y, acc[t][R + (SG + 1) % R]);
                    acc[t][R + (SG + 2) % R] = fmaf(w, tB.z, acc[t][R + (SG + 2) % R]);
                    acc[t][R + (SG + 3) % R] = fmaf(w, tB.w, acc[t][R + (SG + 3) % R]);
                }
            }
        };
        auto fetch = [&](int o) {
            CBCT_DEV_ASSERT(o >= 0 && o < P.t_entries);
            if (R == 4) return __ldg(reinterpret_cast<const float4 *>(T) + o);
            return make_float4(__ldg(T + o), 0.0f, 0.0f, 0.0f);
        };
        // the first two rows together (about two rows cross a voxel): both weights, then all four
        // loads, then the FMAs; a voxel with one row reads it twice with the second weight 0
        {
            const bool two = iv < iv_hi;
            const int ivb = two ? iv + 1 : iv;
            const float w0 = weight(iv), w1 = two ? weight(ivb) : 0.0f;
            const float4 a0 = fetch(oA + iv), a1 = fetch(oA + ivb);
            float4 b0 = a0, b1 = a1;
            if (M == 2) { b0 = fetch(oB - iv); b1 = fetch(oB - ivb); }
            gather(w0, a0, b0);
            gather(w1, a1, b1);
        }
        for (iv += 2; iv <= iv_hi; ++iv) {
            const float w = weight(iv);
            const float4 a0 = fetch(oA + iv);
            float4 b0 = a0;
            if (M == 2) b0 = fetch(oB - iv);
            gather(w, a0, b0);
        }
    }
}

template <int R, int M, int KT>
__global__ void __launch_bounds__(32 * BK_BX, 3)
back_kernel(const LevelParams P, const RayU *__restrict__ rayu, const ViewC *__restrict__ views,
            const float *__restrict__ TL, const float *__restrict__ f, float coef, float *__restrict__ out, int z_off)
{
    const int lane = threadIdx.x;
    const int i = blockIdx.x * BK_BX + threadIdx.y;
    const int j = blockIdx.y;
    const int ni = R == 4 ? P.nx / 2 : P.nx;
    const int nzh = P.nz / M;                        // M == 2: the upper half are the mirror images nz-1-k
    if (i >= ni) return;                             // warp-uniform
    int kv[KT];
    float zl[KT];                                    // lower z-plane of the voxel relative to the source plane (index units)
#pragma unroll
    for (int t = 0; t < KT; ++t) {
        kv[t] = (blockIdx.z + z_off) * (32 * KT) + lane + 32 * t;       // z_off: first z-unit of a sharded launch
        zl[t] = (float)(min(kv[t], nzh - 1) - P.cz) - P.sz;      // a ragged tail recomputes the last voxel, not stored
    }
    // the R quarter-turn images of the voxel: (i,j), (n-1-j, i), (n-1-i, n-1-j), (j, n-1-i)
    int vi[R], vj[R];
    vi[0] = i; vj[0] = j;
    if (R == 4) {
        const int n1 = P.nx - 1;
        vi[1 % R] = n1 - j; vj[1 % R] = i;
        vi[2 % R] = n1 - i; vj[2 % R] = n1 - j;
        vi[3 % R] = j;      vj[3 % R] = n1 - i;
    }
    float acc[KT][R * M];
#pragma unroll
    for (int t = 0; t < KT; ++t)
#pragma unroll
        for (int q = 0; q < R * M; ++q) acc[t][q] = 0.0f;
    const float c0v = -P.v0 * P.inv_dv;
    for (int a = 0; a < P.nbase; ++a) {
        const float4 vw = __ldg(reinterpret_cast<const float4 *>(views) + a);   // c, s, dn, du
#pragma unroll
        for (int sg = 0; sg < R; ++sg) {
            const float xc = fmaf((float)vi[sg], P.hx, P.x0), yc = fmaf((float)vj[sg], P.hy, P.y0);
            const float bx = (float)(vi[sg] - P.cx), by = (float)(vj[sg] - P.cy);
            const float rn = fmaf(xc, vw.x, fmaf(yc, vw.y, P.sad));   // (X - S).e_n  > 0
            const float ru = fmaf(xc, vw.y, -yc * vw.x);               // (X - S).e_u
            // shadow of the (i,j) square on the detector's u axis (Eq. A6): u* = sdd ru/rn to first order in the
            // voxel's half extents dn, du (inflated in the table), plus 0.02 pixel
            float rinv;
            asm("rcp.approx.ftz.f32 %0, %1;" : "=f"(rinv) : "f"(rn));
            const float mag = P.sdd * rinv, tn = ru * rinv;
            const float uc = mag * ru, W = mag * fmaf(fabsf(tn), vw.z, vw.w);
            const int iu_lo = max(0, __float2int_ru((uc - W - P.u0) * P.inv_du - 0.02f));
            const int iu_hi = min(P.nu - 1, __float2int_rd((uc + W - P.u0) * P.inv_du + 0.02f));
            for (int iu = iu_lo; iu <= iu_hi; ++iu) {
                const RayU r = load_rayu(rayu, a * P.nu + iu);
                const float d0 = r.drive ? by : bx, mn = r.drive ? bx : by;   // slab coordinate, minor plane
                // in-plane: t-interval where minor(t) = y0 + t m lies in [mn, mn+1)
                const float y0 = fmaf(d0, r.m, r.a0);
                const float t1 = (mn - y0) * r.inv_m, t2 = (mn + 1.0f - y0) * r.inv_m;
                const float s_lo = fmaxf(fminf(t1, t2), 0.0f), s_hi = fminf(fmaxf(t1, t2), 1.0f);
                if (!(s_hi > s_lo)) continue;
                const float e = d0 - r.sd;                               // slab start relative to the source
                float icA, icB;
                asm("rcp.approx.ftz.f32 %0, %1;" : "=f"(icA) : "f"(r.q * (e + s_lo)));
                asm("rcp.approx.ftz.f32 %0, %1;" : "=f"(icB) : "f"(r.q * (e + s_hi)));
                const float ic_near = fmaxf(icA, icB), ic_far = fminf(icA, icB);     // 1/c at the end nearer to / farther from the source
                const int oA = (a * P.nu + iu) * P.nv;                  // 32-bit entry offset of the column's row 0
                if (sg == 0) gather_column<R, M, KT, 0>(acc, zl, P, TL, c0v, s_lo, s_hi, e, r.q, r.inv_dd, ic_near, ic_far, oA);
                else if (sg == 1) gather_column<R, M, KT, 1 % R>(acc, zl, P, TL, c0v, s_lo, s_hi, e, r.q, r.inv_dd, ic_near, ic_far, oA);
                else if (sg == 2) gather_column<R, M, KT, 2 % R>(acc, zl, P, TL, c0v, s_lo, s_hi, e, r.q, r.inv_dd, ic_near, ic_far, oA);
                else gather_column<R, M, KT, 3 % R>(acc, zl, P, TL, c0v, s_lo, s_hi, e, r.q, r.inv_dd, ic_near, ic_far, oA);
            }
        }
    }
#pragma unroll
    for (int t = 0; t < KT; ++t)
#pragma unroll
        for (int mm = 0; mm < M; ++mm)
#pragma unroll
            for (int q = 0; q < R; ++q) {
                const float v = acc[t][mm * R + q];
                if (kv[t] < nzh) {
                    const size_t o = ((size_t)(mm ? P.nz - 1 - kv[t] : kv[t]) * P.ny + vj[q]) * P.nx + vi[q];
                    out[o] = f ? fmaf(-coef, v, __ldg(f + o)) : v;
                }
            }
}

// The same back-projector with the in-plane part taken out of the warp-uniform instruction stream.  In back_kernel
// every lane of a warp repeats the in-plane arithmetic of its (i,j) (about a fifth of all instructions at 256^3); here
// the lanes of the warp first work through DIFFERENT (base view, voxel image) pairs -- 32 / R base views per round --
// and append the columns that hit to a per-warp list in shared memory (s_lo, s_hi, e, q | 1/c near, 1/c far, inv_dd,
// entry offset), in a fixed order (candidate index, then lane): ballot + popc, no atomics.  Then all lanes walk the
// list (broadcast reads) and gather their KT voxels as before.  A round holds at most BK_MAXC candidate columns per
// pair (checked at launch against the geometry; larger shadows take back_kernel).
constexpr int BK_MAXC = 5, BK_LIST = 32 * BK_MAXC;      // list entries per warp and round (all images together)

template <int R, int M, int KT>
__global__ void __launch_bounds__(32 * BK_BX, 3)
back_list_kernel(const LevelParams P, const RayU *__restrict__ rayu, const ViewC *__restrict__ views,
                 const float *__restrict__ TL, const float *__restrict__ f, float coef, float *__restrict__ out, int z_off)
{
    __shared__ float4 s_list[BK_BX][2][BK_LIST];
    constexpr int LCAP = BK_LIST / R;                 // per image: (32 / R) base views x BK_MAXC
    const int lane = threadIdx.x;
    const int i = blockIdx.x * BK_BX + threadIdx.y;
    const int j = blockIdx.y;
    const int ni = R == 4 ? P.nx / 2 : P.nx;
    const int nzh = P.nz / M;
    if (i >= ni) return;                             // warp-uniform
    float4 *__restrict__ l0 = s_list[threadIdx.y][0], *__restrict__ l1 = s_list[threadIdx.y][1];
    int kv[KT];
    float zl[KT];
#pragma unroll
    for (int t = 0; t < KT; ++t) {
        kv[t] = (blockIdx.z + z_off) * (32 * KT) + lane + 32 * t;       // z_off: first z-unit of a sharded launch
        zl[t] = (float)(min(kv[t], nzh - 1) - P.cz) - P.sz;
    }
    int vi[R], vj[R];
    vi[0] = i; vj[0] = j;
    if (R == 4) {
        const int n1 = P.nx - 1;
        vi[1 % R] = n1 - j; vj[1 % R] = i;
        vi[2 % R] = n1 - i; vj[2 % R] = n1 - j;
        vi[3 % R] = j;      vj[3 % R] = n1 - i;
    }
    float acc[KT][R * M];
#pragma unroll
    for (int t = 0; t < KT; ++t)
#pragma unroll
        for (int q = 0; q < R * M; ++q) acc[t][q] = 0.0f;
    const float c0v = -P.v0 * P.inv_dv;
    // this lane's pair in a round: image my_sg of base view a0 + lane / R
    const int my_sg = lane % R;
    int mi = vi[0], mj = vj[0];
#pragma unroll
    for (int q = 1; q < R; ++q) if (my_sg == q) { mi = vi[q]; mj = vj[q]; }
    const float xc = fmaf((float)mi, P.hx, P.x0), yc = fmaf((float)mj, P.hy, P.y0);
    const float bx = (float)(mi - P.cx), by = (float)(mj - P.cy);
    const unsigned lt_mask = (1u << lane) - 1u;
    const unsigned all_sg = R == 4 ? 0x11111111u : 0xffffffffu;      // lanes that hold image 0
    const unsigned my_mask = all_sg << my_sg;
    for (int a0 = 0; a0 < P.nbase; a0 += 32 / R) {
        int cnt[R];
#pragma unroll
        for (int q = 0; q < R; ++q) cnt[q] = 0;
        const int a = a0 + lane / R;
        int iu_lo = 0, ncand = 0;
        if (a < P.nbase) {
            const float4 vw = __ldg(reinterpret_cast<const float4 *>(views) + a);   // c, s, dn, du
            const float rn = fmaf(xc, vw.x, fmaf(yc, vw.y, P.sad));   // (X - S).e_n  > 0
            const float ru = fmaf(xc, vw.y, -yc * vw.x);               // (X - S).e_u
            float rinv;
            asm("rcp.approx.ftz.f32 %0, %1;" : "=f"(rinv) : "f"(rn));
            const float mag = P.sdd * rinv, tn = ru * rinv;
            const float uc = mag * ru, W = mag * fmaf(fabsf(tn), vw.z, vw.w);
            iu_lo = max(0, __float2int_ru((uc - W - P.u0) * P.inv_du - 0.02f));
            const int iu_hi = min(P.nu - 1, __float2int_rd((uc + W - P.u0) * P.inv_du + 0.02f));
            CBCT_DEV_ASSERT(iu_hi - iu_lo + 1 <= BK_MAXC);       // the bound checked at create (Level::back_maxc)
            ncand = min(iu_hi - iu_lo + 1, BK_MAXC);
        }
        for (int c = 0; __any_sync(0xffffffffu, c < ncand); ++c) {
            bool ok = c < ncand;
            float4 e0 = make_float4(0.f, 0.f, 0.f, 0.f), e1 = e0;
            if (ok) {
                const int iu = iu_lo + c;
                const RayU r = load_rayu(rayu, a * P.nu + iu);
                const float d0 = r.drive ? by : bx, mn = r.drive ? bx : by;   // slab coordinate, minor plane
                const float y0 = fmaf(d0, r.m, r.a0);
                const float t1 = (mn - y0) * r.inv_m, t2 = (mn + 1.0f - y0) * r.inv_m;
                const float s_lo = fmaxf(fminf(t1, t2), 0.0f), s_hi = fminf(fmaxf(t1, t2), 1.0f);
                ok = s_hi > s_lo;
                const float e = d0 - r.sd;
                float icA, icB;
                asm("rcp.approx.ftz.f32 %0, %1;" : "=f"(icA) : "f"(r.q * (e + s_lo)));
                asm("rcp.approx.ftz.f32 %0, %1;" : "=f"(icB) : "f"(r.q * (e + s_hi)));
                e0 = make_float4(s_lo, s_hi, e, r.q);
                e1 = make_float4(fmaxf(icA, icB), fminf(icA, icB), r.inv_dd, __int_as_float((a * P.nu + iu) * P.nv));
            }
            const unsigned hit = __ballot_sync(0xffffffffu, ok);
            if (ok) {
                int my_cnt = cnt[0];
#pragma unroll
                for (int q = 1; q < R; ++q) if (my_sg == q) my_cnt = cnt[q];
                const int pos = my_sg * LCAP + my_cnt + __popc(hit & my_mask & lt_mask);
                CBCT_DEV_ASSERT(pos >= my_sg * LCAP && pos < (my_sg + 1) * LCAP);
                l0[pos] = e0; l1[pos] = e1;
            }
#pragma unroll
            for (int q = 0; q < R; ++q) cnt[q] += __popc(hit & (all_sg << q));
        }
        __syncwarp();
#pragma unroll
        for (int sg = 0; sg < R; ++sg) {
            for (int n = 0; n < cnt[sg]; ++n) {
                const float4 e0 = l0[sg * LCAP + n], e1 = l1[sg * LCAP + n];
                const int oA = __float_as_int(e1.w);
                if (sg == 0) gather_column<R, M, KT, 0>(acc, zl, P, TL, c0v, e0.x, e0.y, e0.z, e0.w, e1.z, e1.x, e1.y, oA);
                else if (sg == 1) gather_column<R, M, KT, 1 % R>(acc, zl, P, TL, c0v, e0.x, e0.y, e0.z, e0.w, e1.z, e1.x, e1.y, oA);
                else if (sg == 2) gather_column<R, M, KT, 2 % R>(acc, zl, P, TL, c0v, e0.x, e0.y, e0.z, e0.w, e1.z, e1.x, e1.y, oA);
                else gather_column<R, M, KT, 3 % R>(acc, zl, P, TL, c0v, e0.x, e0.y, e0.z, e0.w, e1.z, e1.x, e1.y, oA);
            }
        }
        __syncwarp();
    }
#pragma unroll
    for (int t = 0; t < KT; ++t)
#pragma unroll
        for (int mm = 0; mm < M; ++mm)
#pragma unroll
            for (int q = 0; q < R; ++q) {
                const float v = acc[t][mm * R + q];
                if (kv[t] < nzh) {
                    const size_t o = ((size_t)(mm ? P.nz - 1 - kv[t] : kv[t]) * P.ny + vj[q]) * P.nx + vi[q];
                    out[o] = f ? fmaf(-coef, v, __ldg(f + o)) : v;
                }
            }
}

template <int R, int M, int KT>
static void launch_back_kernel(const LevelParams &P, const Level &L, const float *src, const float *d_f, float coef,
                               float *d_out, cudaStream_t st, const Shard *sh)
{
    const int nzh = P.nz / M, ni = R == 4 ? P.nx / 2 : P.nx, nj = R == 4 ? P.ny / 2 : P.ny;
    const int kchunk = 32 * KT;
    dim3 b(32, BK_BX), gr((ni + BK_BX - 1) / BK_BX, nj, (nzh + kchunk - 1) / kchunk);
    int z_off = 0;
    if (sh) { z_off = sh->zu_lo; gr.z = sh->zu_hi - sh->zu_lo; if (gr.z == 0) return; }
    if (L.back_maxc <= BK_MAXC) back_list_kernel<R, M, KT><<<gr, b, 0, st>>>(P, L.d_rayu, L.d_view, src, d_f, coef, d_out, z_off);
    else back_kernel<R, M, KT><<<gr, b, 0, st>>>(P, L.d_rayu, L.d_view, src, d_f, coef, d_out, z_off);
}

// voxels per thread along z: two at 80 registers measured best at 256^3 (1 and 4 voxels, 64 / 100+ registers: 3-50 % slower)
static int back_kt(const LevelParams &P) { return P.nz / P.nmir >= 64 ? 2 : 1; }

template <int R, int M>
static void launch_back_rm(const LevelParams &P, const Level &L, const float *src, const float *d_f, float coef,
                           float *d_out, cudaStream_t st, const Shard *sh)
{
    if (back_kt(P) == 2) launch_back_kernel<R, M, 2>(P, L, src, d_f, coef, d_out, st, sh);
    else launch_back_kernel<R, M, 1>(P, L, src, d_f, coef, d_out, st, sh);
}

// The z-unit of a sharded back-projection: the slices one block of the level's kernel covers along z.
int back_zunit(const Level &L) { return L.bt.ok ? 32 * L.bt.ZV : 32 * back_kt(L.p); }
int back_nzunits(const Level &L)
{
    const int nzh = L.p.nz / L.p.nmir, u = back_zunit(L);
    return (nzh + u - 1) / u;
}

cbct_status launch_back(const cbct_geometry *g, const Level &L, const float *d_in, int scaled,
                        const float *d_f, float coef, float *d_out, cudaStream_t st, const Shard *sh)
{
    const LevelParams &P = L.p;
    const float *src = d_in;
    if (L.bt.ok && scaled && d_in != L.d_T)
        return cbct_fail(CBCT_ERR_INVALID_ARG, "launch_back: the TMA path reads the level's own residual stack");
    if (!scaled) {
        StageTimer t(g, st, ST_TRANSFER);
        dim3 b(128), gr((P.nu + 127) / 128, P.nv, P.nbase);
        if (P.nsym == 4) scale_by_L_kernel<4><<<gr, b, 0, st>>>(P, L.d_rayu, d_in, L.d_T);
        else scale_by_L_kernel<1><<<gr, b, 0, st>>>(P, L.d_rayu, d_in, L.d_T);
        CBCT_LAUNCH_CHECK(g);
        src = L.d_T;
    }
    StageTimer t(g, st, ST_BACK);
    if (sh && (sh->zu_lo < 0 || sh->zu_hi > back_nzunits(L) || sh->zu_lo > sh->zu_hi)) return cbct_fail(CBCT_ERR_INVALID_ARG, "launch_back: bad shard");
    if (L.bt.ok) return launch_back_tma(g, L, d_f, coef, d_out, st, sh);      // src is L.d_T on this path (below)
    if (P.nsym == 4 && P.nmir == 2) launch_back_rm<4, 2>(P, L, src, d_f, coef, d_out, st, sh);
    else if (P.nsym == 4) launch_back_rm<4, 1>(P, L, src, d_f, coef, d_out, st, sh);
    else if (P.nmir == 2) launch_back_rm<1, 2>(P, L, src, d_f, coef, d_out, st, sh);
    else launch_back_rm<1, 1>(P, L, src, d_f, coef, d_out, st, sh);
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
