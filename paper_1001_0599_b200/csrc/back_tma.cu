// back_tma.cu -- A3/A4: the exact-transpose back-projector on TMA + shared memory (sm_100a).
//
// Same operator as back.cu -- (P^T T)[voxel] = sum_views sum_rays len(ray ∩ voxel) T[ray] with the coefficients of
// forward.cu ("sum_theta P^T (P f - Y)"; the paper itself evaluates the continuum adjoint Eq. 6,
// L195-L199, because a scatter collides on voxels, L187-L191) -- and the same arithmetic per (ray, voxel) pair (ray.cuh),
// with the residual stack moved off the L1/LSU path:
//
//  * A block owns a BRICK of BI x BJ voxel columns of the first quadrant and 32 z-slices of the lower half of the
//    volume, together with their quarter-turn and mirror images (8 voxels per weight, back.cu).  A warp owns CPW of the
//    brick's columns; its lanes run along z.
//  * The work is cut into STAGES (base view a, voxel image sg).  For one stage the brick casts a compact shadow on
//    the detector of the base view: a few columns x the rows its 32 slices reach (exactly those rows again, mirrored,
//    for the upper half of the volume).  A producer warp computes that rectangle and has the TMA unit copy it from the
//    quarter-turn-interleaved residual stack (16-byte entries, detector rows fastest) into a ring of shared-memory tiles:
//    one `cp.async.bulk.tensor` per power-of-two group of columns, completion counted on an mbarrier, rows outside the
//    detector zero-filled by the copy unit -- so the gather loop holds no range clamp and no global load.
//  * The consumer warps wait on the tile's "full" barrier, gather from shared memory and release the tile through its
//    "empty" barrier; the producer runs one stage ahead, so the L2 round trips the L1-path kernel waited on (35 %
//    occupancy, profiles/r01d) overlap the arithmetic of the previous stage.
//  * About two detector rows cross a voxel, so consecutive lanes read 16-byte entries ~2 rows apart: in a plain layout
//    that is a two-way bank conflict on every load.  The residual stack is therefore stored split by row parity
//    (LevelParams::tP == 2: even rows, then odd rows of a column) and the odd plane of a tile is shifted by one entry,
//    which puts rows r and r + 2 in adjacent 16-byte bank groups and rows r, r + 1 apart.
//  * The in-plane part of every (column of voxels, base view, image, detector column) is worked out once per warp by
//    lanes in parallel, as in back_list_kernel, into a per-warp list; the rows of a voxel start at an exact first row
//    and take a fixed number NSLOT of slots (a bound from the geometry, checked at create): rows past the voxel get
//    weight 0 from the same clipping that computes every weight, and the last slot's loads are predicated on it.
//  * The 8 x 32 x BI x BJ results of a brick go through shared memory once more and leave in x-fastest order with
//    16-byte stores (fused with g = f - coef * b, A4).
//
// Summation order per voxel: base view, image, detector column, row -- fixed, no atomics: bitwise reproducible.
#include <cuda.h>
#include <math.h>
#include "cbct_internal.cuh"
#include "ray.cuh"

namespace {

__device__ __forceinline__ uint32_t smem_u32(const void *p) { return (uint32_t)__cvta_generic_to_shared(p); }

__device__ __forceinline__ void mbar_init(uint32_t bar, uint32_t count)
{
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(bar), "r"(count) : "memory");
}
__device__ __forceinline__ void mbar_arrive(uint32_t bar)
{
    asm volatile("{\n .reg .b64 st;\n mbarrier.arrive.shared::cta.b64 st, [%0];\n}" ::"r"(bar) : "memory");
}
__device__ __forceinline__ void mbar_arrive_expect_tx(uint32_t bar, uint32_t bytes)
{
    asm volatile("{\n .reg .b64 st;\n mbarrier.arrive.expect_tx.shared::cta.b64 st, [%0], %1;\n}" ::"r"(bar), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_wait(uint32_t bar, uint32_t parity)
{
    asm volatile(
        "{\n"
        " .reg .pred p;\n"
        "BT_WAIT:\n"
        " mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n"
        " @p bra BT_DONE;\n"
        " bra BT_WAIT;\n"
        "BT_DONE:\n"
        "}" ::"r"(bar), "r"(parity) : "memory");
}
// one box of the 4-d view (row pair index within a plane, plane, detector column, base view) of the residual stack
__device__ __forceinline__ void tma_load_4d(uint32_t dst, const CUtensorMap *map, int c0, int c1, int c2, int c3, uint32_t bar)
{
    asm volatile("cp.async.bulk.tensor.4d.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1, {%2, %3, %4, %5}], [%6];"
                 ::"r"(dst), "l"(reinterpret_cast<uint64_t>(map)), "r"(c0), "r"(c1), "r"(c2), "r"(c3), "r"(bar) : "memory");
}

__device__ __forceinline__ float rcp_approx(float x)
{
    float r;
    asm("rcp.approx.ftz.f32 %0, %1;" : "=f"(r) : "f"(x));
    return r;
}

// image sg of the first-quadrant voxel (i, j) under quarter turns: (i,j), (n1-j, i), (n1-i, n1-j), (j, n1-i)
__device__ __forceinline__ void bt_image(int sg, int i, int j, int n1, int &mi, int &mj)
{
    mi = sg == 0 ? i : sg == 1 ? n1 - j : sg == 2 ? n1 - i : j;
    mj = sg == 0 ? j : sg == 1 ? i : sg == 2 ? n1 - j : n1 - i;
}

// Shadow of the (mi, mj) voxel square on the u axis of base view `vw` (Eq. A6, to first order in the inflated
// half extents; the expressions of back.cu): detector columns [iu_lo, iu_hi], and the voxel centre's depth rn along e_n.
__device__ __forceinline__ void bt_shadow(const LevelParams &P, const float4 vw, int mi, int mj, int &iu_lo, int &iu_hi, float &rn)
{
    const float xc = fmaf((float)mi, P.hx, P.x0), yc = fmaf((float)mj, P.hy, P.y0);
    rn = fmaf(xc, vw.x, fmaf(yc, vw.y, P.sad));
    const float ru = fmaf(xc, vw.y, -yc * vw.x);
    const float rinv = rcp_approx(rn);
    const float mag = P.sdd * rinv, tn = ru * rinv;
    const float uc = mag * ru, W = mag * fmaf(fabsf(tn), vw.z, vw.w);
    iu_lo = max(0, __float2int_ru((uc - W - P.u0) * P.inv_du - 0.02f));
    iu_hi = min(P.nu - 1, __float2int_rd((uc + W - P.u0) * P.inv_du + 0.02f));
}

__device__ __forceinline__ float4 lds128(uint32_t addr)
{
    float4 v;
    asm volatile("ld.shared.v4.f32 {%0, %1, %2, %3}, [%4];" : "=f"(v.x), "=f"(v.y), "=f"(v.z), "=f"(v.w) : "r"(addr));
    return v;
}

// One detector column's contribution to a voxel and its 7 images.  e0 = (s_lo, s_hi, e, q), e1 = (-, 1/c at the
// strip end nearer to the source in detector rows per z-index, the column's shared-memory address in the stage's A tile,
// oA) with s_lo, s_hi, e, q as in back.cu.  The voxel lies below the source plane (zlo + 1 <= 0): its rows have v < 0, so
// its two z-planes are crossed in a known order -- plane zlo + oA first, oA = 1 when q > 0 -- and rows with v > 0 clip to
// weight 0 by the same expressions.  A lane whose rows all lie below the detector (the
// truncated bottom of the volume) does nothing.
// The in-plane part of (voxel column (vi0, vj0) of the first quadrant, base view, image sg, candidate detector column cnd of the
// image's shadow): e0 = (s_lo, s_hi, e, q), e1 = (-, 1/c, -, oA) as bt_visit reads them, and the detector column iu.  One
// definition for the list rounds of the kernel and for the table built once per geometry (bt_build_lists_kernel): the two
// hold the same bits.
__device__ __forceinline__ bool bt_list_entry(const LevelParams &P, const float4 vw, const RayU *__restrict__ rayu, int a, int vi0,
                                              int vj0, int n1, int sg, int cnd, float4 &e0, float4 &e1, int &iu)
{
    int mi, mj, iu_lo, iu_hi;
    float rn;
    bt_image(sg, vi0, vj0, n1, mi, mj);
    bt_shadow(P, vw, mi, mj, iu_lo, iu_hi, rn);
    CBCT_DEV_ASSERT(iu_hi - iu_lo + 1 <= BT_MAXC);
    if (cnd > iu_hi - iu_lo) return false;
    iu = iu_lo + cnd;
    const RayU r = load_rayu(rayu, a * P.nu + iu);
    const float bx = (float)(mi - P.cx), by = (float)(mj - P.cy);
    const float d0 = r.drive ? by : bx, mn = r.drive ? bx : by;
    const float y0 = fmaf(d0, r.m, r.a0);
    const float t1 = (mn - y0) * r.inv_m, t2 = (mn + 1.0f - y0) * r.inv_m;
    const float s_lo = fmaxf(fminf(t1, t2), 0.0f), s_hi = fminf(fmaxf(t1, t2), 1.0f);
    const float e = d0 - r.sd;
    const float icA = rcp_approx(r.q * (e + s_lo)), icB = rcp_approx(r.q * (e + s_hi));
    e0 = make_float4(s_lo, s_hi, e, r.q);
    e1 = make_float4(0.0f, fmaxf(icA, icB) * P.inv_dv, 0.0f, r.q > 0.0f ? 1.0f : 0.0f);
    return s_hi > s_lo;
}

// The list table: for every first-quadrant voxel column and base view, BT_TABH entries per image in candidate order
// (32 float4 = 512 bytes: entry (sg, n) at float4 2 (4 sg + n) and the next), the count of an image in the .x of its first
// entry's second half, the detector column in the .z.  One warp per (column, base view); *overflow counts images with more hits.
constexpr int BT_TABH = 4;
__global__ void bt_build_lists_kernel(const LevelParams P, const RayU *__restrict__ rayu, const ViewC *__restrict__ views,
                                      float4 *__restrict__ table, unsigned int *__restrict__ overflow)
{
    const int lane = threadIdx.x & 31, w = blockIdx.x * (blockDim.x >> 5) + (threadIdx.x >> 5);
    const int ni = P.nx / 2, nj = P.ny / 2;
    if (w >= ni * nj * P.nbase) return;
    const int a = w % P.nbase, colidx = w / P.nbase, vi0 = colidx % ni, vj0 = colidx / ni;
    const float4 vw = __ldg(reinterpret_cast<const float4 *>(views) + a);
    const int sg = lane >> 3, cnd = lane & 7;
    float4 e0 = make_float4(0.f, 0.f, 0.f, 0.f), e1 = e0;
    int iu = 0;
    const bool ok = bt_list_entry(P, vw, rayu, a, vi0, vj0, P.nx - 1, sg, cnd, e0, e1, iu);
    const unsigned hit = __ballot_sync(0xffffffffu, ok);
    const unsigned grp = hit & (0xffu << (8 * sg));
    const int rank = __popc(grp & ((1u << lane) - 1u)), cnt = __popc(grp);
    if (cnt > BT_TABH && cnd == 0) atomicAdd(overflow, 1u);
    if (ok && rank < BT_TABH) {
        e1.z = __int_as_float(iu);
        if (rank == 0) e1.x = __int_as_float(cnt);
        float4 *t = table + (size_t)w * 32 + 2 * (BT_TABH * sg + rank);
        t[0] = e0; t[1] = e1;
    }
}

template <int SG, int NSLOT, int TP, int ZV>
__device__ __forceinline__ void bt_visit(float (&acc)[ZV][8], const BtConsts &C, const float (&zlo)[ZV], const float4 e0, const float4 e1,
                                         int r0A)
{
    int r[ZV];
    bool any = false;
#pragma unroll
    for (int v = 0; v < ZV; ++v) {
        r[v] = __float2int_ru(fmaf(zlo[v], e1.y, C.c0v_m));
        any = any || r[v] + NSLOT > 0;
    }
    if (!any) return;                   // every row of this lane's voxels lies below the detector (zero-filled rows otherwise)
    const float e = e0.z;
    const uint32_t colA = (uint32_t)__float_as_int(e1.z);
    float w[ZV][NSLOT];
    uint32_t aA[ZV], aB[ZV], d1[ZV];
#pragma unroll
    for (int v = 0; v < ZV; ++v) {
        const int rr = r[v] - r0A;
        CBCT_DEV_ASSERT(rr >= 0 && rr + NSLOT - 1 <= C.rr_max);
        const float zA = zlo[v] + e1.w, zB = zlo[v] + 1.0f - e1.w;
        // byte offset of row rr in its column: rr / 2 entries into the plane of its parity, the odd plane shifted by one entry
        uint32_t off;
        if (TP == 2) {
            const int p = rr & 1;
            off = rr * 8 + p * C.plane_step8;              // (rr >> 1) * 16 + p * (plane_bytes + 16)
            d1[v] = p ? C.step_odd : C.step_even;          // to row rr + 1: the other plane
        } else {
            off = rr << 4;
            d1[v] = 16;
        }
        aA[v] = colA + off; aB[v] = colA + C.KB - off;
        const float rf = (float)r[v];
#pragma unroll
        for (int s = 0; s < NSLOT; ++s) {
            // v from one rounding of r dv + v0 (it cancels to a fraction of a pixel at the centre of the detector, and the
            // crossing parameter amplifies its relative error by the source distance in slabs); v != 0: even row count, centred
            const float inv = rcp_approx(fmaf(rf + (float)s, C.dv, C.v0) * e0.w);
            const float qa = fmaf(zA, inv, -e), qb = fmaf(zB, inv, -e);
            w[v][s] = fmaxf(fminf(qb, e0.y) - fmaxf(qa, e0.x), 0.0f);
        }
    }
#pragma unroll
    for (int s = 0; s < NSLOT; ++s) {
#pragma unroll
        for (int v = 0; v < ZV; ++v) {
            const uint32_t os = TP == 2 ? (s & 1) * d1[v] + (s >> 1) * 16 : 16 * s;
            if (s < NSLOT - 1 || w[v][s] > 0.0f) {
                const float4 tA = lds128(aA[v] + os);
                const float4 tB = lds128(aB[v] - os);
                const float ww = w[v][s];
                acc[v][(SG + 0) % 4] = fmaf(ww, tA.x, acc[v][(SG + 0) % 4]);
                acc[v][(SG + 1) % 4] = fmaf(ww, tA.y, acc[v][(SG + 1) % 4]);
                acc[v][(SG + 2) % 4] = fmaf(ww, tA.z, acc[v][(SG + 2) % 4]);
                acc[v][(SG + 3) % 4] = fmaf(ww, tA.w, acc[v][(SG + 3) % 4]);
                acc[v][4 + (SG + 0) % 4] = fmaf(ww, tB.x, acc[v][4 + (SG + 0) % 4]);
                acc[v][4 + (SG + 1) % 4] = fmaf(ww, tB.y, acc[v][4 + (SG + 1) % 4]);
                acc[v][4 + (SG + 2) % 4] = fmaf(ww, tB.z, acc[v][4 + (SG + 2) % 4]);
                acc[v][4 + (SG + 3) % 4] = fmaf(ww, tB.w, acc[v][4 + (SG + 3) % 4]);
            }
        }
    }
}

// Detector rectangle of one stage (base view of vw, image sg) of the brick at (i0, j0), slices k0 .. k0 + 32 ZV - 1: header =
// (skip, first detector column, first row of the A window, columns).  Warp-collective; one definition for the kernel and for
// the table built once per geometry (bt_build_headers_kernel).  Bounds of create that do not hold are counted in *errflag.
template <int BI, int BJ, int NSLOT, int TP, int ZV>
__device__ __forceinline__ int4 bt_stage_header(const LevelParams &P, const BtParams &Q, const float4 vw, int i0, int j0, int k0, int sg,
                                                int lane, unsigned int *errflag)
{
    constexpr int NIJ = BI * BJ;
    const int ni = P.nx / 2, nj = P.ny / 2, n1 = P.nx - 1;
    const int rr_max = TP * Q.XB - (TP == 2 ? 3 : 1);
    int cmin = 1 << 30, cmax = -1;
    float rn_lo = 3.0e38f, rn_hi = -3.0e38f;
    for (int v = lane; v < NIJ; v += 32) {
        const int i = i0 + v % BI, j = j0 + v / BI;
        if (i < ni && j < nj) {
            int mi, mj, lo, hi;
            float rn;
            bt_image(sg, i, j, n1, mi, mj);
            bt_shadow(P, vw, mi, mj, lo, hi, rn);
            if (lo <= hi) { cmin = min(cmin, lo); cmax = max(cmax, min(hi, lo + BT_MAXC - 1)); }
            rn_lo = fminf(rn_lo, rn); rn_hi = fmaxf(rn_hi, rn);
        }
    }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) {
        cmin = min(cmin, __shfl_xor_sync(0xffffffffu, cmin, o));
        cmax = max(cmax, __shfl_xor_sync(0xffffffffu, cmax, o));
        rn_lo = fminf(rn_lo, __shfl_xor_sync(0xffffffffu, rn_lo, o));
        rn_hi = fmaxf(rn_hi, __shfl_xor_sync(0xffffffffu, rn_hi, o));
    }
    // rows: v = z hz sdd / rn for a point at depth rn; the strip ends of a voxel lie within its half extent dn
    // (vw.z, inflated) of its centre's depth.  First row of the lowest slice, last slot of the highest.
    const int klast = min(k0 + 32 * ZV - 1, Q.nzh - 1);
    const float zf = (float)(k0 - P.cz) - P.sz, zl = (float)(klast - P.cz) - P.sz;
    const float ic_max = Q.ic_scale / (rn_lo - vw.z) * 1.00001f, ic_min = Q.ic_scale / (rn_hi + vw.z) * 0.99999f;
    const int rmin = __float2int_ru(fmaf(zf, ic_max, Q.c0v_m)) - 1;
    const int rlast = __float2int_ru(fmaf(zl, ic_min, Q.c0v_m)) + NSLOT;
    int ncols = cmax - cmin + 1;
    const bool skip = ncols <= 0 || rlast < 0 || rmin > P.nv - 1;
    const int x0 = TP == 2 ? (rmin >> 1) : rmin, r0A = TP * x0;
    if (!skip && (ncols > Q.ncols || rlast - r0A > rr_max)) {   // the bounds of create do not hold: flag, stay in bounds
        if (lane == 0) atomicAdd(errflag, 1u);
        ncols = min(ncols, Q.ncols);
    }
    return make_int4(skip ? 1 : 0, cmin, r0A, ncols);
}

// The header table: [z-unit][brick row][brick column][stage], one warp per header.
template <int BI, int BJ, int NSLOT, int TP, int ZV>
__global__ void bt_build_headers_kernel(const LevelParams P, const BtParams Q, const ViewC *__restrict__ views, int gx, int gy, int gz,
                                        int4 *__restrict__ table, unsigned int *__restrict__ errflag)
{
    const int lane = threadIdx.x & 31;
    const long long w = (long long)blockIdx.x * (blockDim.x >> 5) + (threadIdx.x >> 5);
    const int n_stages = 4 * P.nbase;
    if (w >= (long long)gx * gy * gz * n_stages) return;
    const int s = (int)(w % n_stages);
    const long long b = w / n_stages;
    const int bx = (int)(b % gx), by = (int)((b / gx) % gy), zu = (int)(b / ((long long)gx * gy));
    const float4 vw = __ldg(reinterpret_cast<const float4 *>(views) + (s >> 2));
    const int4 h = bt_stage_header<BI, BJ, NSLOT, TP, ZV>(P, Q, vw, bx * BI, by * BJ, zu * 32 * ZV, s & 3, lane, errflag);
    if (lane == 0) table[w] = h;
}

// R == 4, M == 2 only (square centred in-plane grid with quarter-turn views, volume and detector centred in z / v).
// ZV = voxels per lane along z: a block owns 32 ZV slices of the lower half volume (lane l: slices k0 + l, k0 + 32 + l).  With
// ZV = 2 the in-plane lists, the stage headers and the 4 n_base barrier handshakes of a block serve twice the voxels.
// LT: the in-plane lists come from the table bt_build_lists_kernel made at create (copied into the warp's list area by cp.async,
// one base view ahead of the stages that read them) instead of being worked out by the lanes at the start of every base view.
template <int BI, int BJ, int CPW, int NSLOT, int TP, int MINB, int ZV, bool LT>
__global__ void __launch_bounds__((BI * BJ / CPW + 1) * 32, MINB)
back_tma_kernel(const __grid_constant__ BtMaps maps, const LevelParams P, const BtParams Q,
                const RayU *__restrict__ rayu, const ViewC *__restrict__ views, const float *__restrict__ f, float coef,
                float *__restrict__ out, unsigned int *__restrict__ errflag, int kb_top, const float4 *__restrict__ lists,
                const int4 *__restrict__ hdrs)
{
    constexpr int NIJ = BI * BJ, NW = NIJ / CPW;      // voxel columns of the brick, consumer warps
    constexpr int SPR = 4 / CPW;                      // stages per list round: 32 lanes = SPR stages x CPW columns x 8 candidates
    static_assert(CPW == 1 || CPW == 2 || CPW == 4, "a list round is 32 lanes");
    extern __shared__ __align__(1024) char smem[];
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    // within a brick the slices nearest to the central plane first (the truncated bottom units are the cheap ones)
    constexpr int ZPB = 32 * ZV;                       // slices per block
    // Q.zu_fast: grid = (z-units, bricks in i, bricks in j) -- the z-units of a brick are neighbours in launch order, run at the
    // same time and share the brick's list-table lines in L2 (with the z-unit slowest every unit re-reads the table from DRAM:
    // 445 MB of DRAM reads per launch at config 3, 218 MB so).  Where the residual stack itself does not fit L2 (360 views of
    // 512 x 384: 283 MB) the z-unit stays the slowest index, so that the blocks in flight share one band of detector rows.
    const bool zf = Q.zu_fast != 0;
    const int bz = zf ? blockIdx.x : blockIdx.z, bx = zf ? blockIdx.y : blockIdx.x, by = zf ? blockIdx.z : blockIdx.y;
    const int gx = zf ? gridDim.y : gridDim.x, gy = zf ? gridDim.z : gridDim.y;
    const int i0 = bx * BI, j0 = by * BJ, k0 = (kb_top - 1 - bz) * ZPB;     // kb_top: one past the last z-unit of this launch
    const int ni = P.nx / 2, nj = P.ny / 2, n1 = P.nx - 1;
    const int n_stages = 4 * P.nbase;

    float4 *s_view = reinterpret_cast<float4 *>(smem + Q.view_off);
    int4 *s_hdr = reinterpret_cast<int4 *>(smem + Q.hdr_off);
    const uint32_t bar0 = smem_u32(smem + Q.bar_off);             // full[0], full[1], empty[0], empty[1]
    for (int a = threadIdx.x; a < P.nbase; a += blockDim.x) s_view[a] = __ldg(reinterpret_cast<const float4 *>(views) + a);
    if (threadIdx.x == 0) {
        for (int s = 0; s < BT_NST; ++s) { mbar_init(bar0 + 8 * s, 1); mbar_init(bar0 + 8 * (BT_NST + s), NW); }
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    __syncthreads();

    BtConsts C;
    C.c0v_m = Q.c0v_m; C.dv = P.dv; C.v0 = P.v0; C.rr_max = TP * Q.XB - (TP == 2 ? 3 : 1);
    C.plane_step8 = Q.plane_bytes + 8;
    C.step_even = Q.plane_bytes + 16; C.step_odd = 16 - (Q.plane_bytes + 16);
    C.KB = Q.half_bytes + (TP == 2 ? Q.plane_bytes : 0) + (Q.XB - 1) * 16;

    float acc[CPW][ZV][8];
#pragma unroll
    for (int cp = 0; cp < CPW; ++cp)
#pragma unroll
        for (int v = 0; v < ZV; ++v)
#pragma unroll
            for (int q = 0; q < 8; ++q) acc[cp][v][q] = 0.0f;

    // ---------------- every stage's detector rectangle: from the table made at create, or by all warps, before the ring starts ----
    if (LT && hdrs) {
        const int4 *hb = hdrs + ((size_t)((kb_top - 1 - bz) * gy + by) * gx + bx) * n_stages;
        for (int s = threadIdx.x; s < n_stages; s += blockDim.x) s_hdr[s] = __ldg(hb + s);
    } else {
        for (int s = warp; s < n_stages; s += NW + 1) {
            const int4 h = bt_stage_header<BI, BJ, NSLOT, TP, ZV>(P, Q, s_view[s >> 2], i0, j0, k0, s & 3, lane, errflag);
            if (lane == 0) s_hdr[s] = h;
        }
    }
    __syncthreads();

    if (warp == NW) {
        // ---------------- producer: the tile copies, one stage ahead of the consumers ----------------
        if (lane == 0) {
            for (int s = 0; s < n_stages; ++s) {
                const int a = s >> 2, slot = s % BT_NST, use = s / BT_NST;
                if (use > 0) mbar_wait(bar0 + 8 * (BT_NST + slot), (use - 1) & 1);
                const int4 hdr = s_hdr[s];
                const uint32_t full = bar0 + 8 * slot;
                if (hdr.x) { mbar_arrive(full); continue; }
                const int cmin = hdr.y, ncols = hdr.w, x0 = hdr.z / TP;
                const uint32_t tile = smem_u32(smem + slot * Q.stage_bytes);
                const uint32_t col_bytes = Q.XB * 16;
                mbar_arrive_expect_tx(full, (uint32_t)(2 * TP * ncols) * col_bytes);
                int c = 0;
#pragma unroll
                for (int b = BT_NMAPS - 1; b >= 0; --b) {
                    if (ncols & (1 << b)) {
                        const uint32_t dst = tile + c * col_bytes;
                        if (TP == 2) {
                            const int xb1 = P.nv / 2 - x0 - Q.XB;      // origin of the mirror rows' odd plane
                            tma_load_4d(dst, &maps.m[b], 2 * x0, 0, cmin + c, a, full);
                            tma_load_4d(dst + Q.plane_bytes, &maps.m[b], 2 * (x0 - 1), 1, cmin + c, a, full);
                            tma_load_4d(dst + Q.half_bytes, &maps.m[b], 2 * (xb1 + 1), 0, cmin + c, a, full);
                            tma_load_4d(dst + Q.half_bytes + Q.plane_bytes, &maps.m[b], 2 * xb1, 1, cmin + c, a, full);
                        } else {
                            tma_load_4d(dst, &maps.m[b], 2 * x0, 0, cmin + c, a, full);
                            tma_load_4d(dst + Q.half_bytes, &maps.m[b], 2 * (P.nv - x0 - Q.XB), 0, cmin + c, a, full);
                        }
                        c += 1 << b;
                    }
                }
            }
        }
    } else {
        // ---------------- consumers ----------------
        float4 *__restrict__ l0 = reinterpret_cast<float4 *>(smem + Q.list_off) + warp * 64, *__restrict__ l1 = l0 + 32;
        float zlo[ZV];
#pragma unroll
        for (int v = 0; v < ZV; ++v) zlo[v] = (float)(min(k0 + 32 * v + lane, Q.nzh - 1) - P.cz) - P.sz;
        uint32_t tile0 = smem_u32(smem);
        asm volatile("" : "+r"(tile0));                 // keep the window address in a register
        // this lane's candidate in a list round: unit u = lane / 8 -> (stage of the round, column of the warp), candidate lane % 8
        const int u = lane >> 3, cnd = lane & 7;
        const int my_cp = u % CPW, my_t = u / CPW;
        const int col = warp * CPW + my_cp;
        const int vi0 = i0 + col % BI, vj0 = j0 + col / BI;
        const bool col_ok = vi0 < ni && vj0 < nj;
        const unsigned lt_mask = (1u << lane) - 1u;
        if constexpr (LT) {
            static_assert(CPW == 1, "the list table holds one voxel column per warp");
            // ---- lists from the table: 512 bytes per (column, base view), one 16-byte cp.async per lane, a base view ahead ----
            const float4 *tab = lists + ((size_t)(vj0 * ni + vi0) * P.nbase) * 32 + lane;
            const uint32_t lbuf = smem_u32(l0) + lane * 16;
            if (col_ok) asm volatile("cp.async.cg.shared.global [%0], [%1], 16;" ::"r"(lbuf), "l"(tab) : "memory");
            asm volatile("cp.async.commit_group;" ::: "memory");
            for (int a = 0; a < P.nbase; ++a) {
                if (col_ok && a + 1 < P.nbase)
                    asm volatile("cp.async.cg.shared.global [%0], [%1], 16;" ::"r"(lbuf + ((a + 1) & 1) * 512), "l"(tab + (size_t)(a + 1) * 32) : "memory");
                asm volatile("cp.async.commit_group;" ::: "memory");
                asm volatile("cp.async.wait_group 1;" ::: "memory");
                __syncwarp();
                const float4 *__restrict__ L = l0 + (a & 1) * 32;
#pragma unroll
                for (int sg = 0; sg < 4; ++sg) {
                    const int s = 4 * a + sg, slot = s % BT_NST, use = s / BT_NST;
                    mbar_wait(bar0 + 8 * slot, use & 1);
                    const int4 hdr = s_hdr[s];
                    if (!hdr.x && col_ok) {
                        const int n_u = __float_as_int(L[2 * BT_TABH * sg + 1].x);
                        const uint32_t col0 = tile0 + slot * Q.stage_bytes - hdr.y * (Q.XB * 16);
                        for (int n = 0; n < n_u; ++n) {
                            const float4 E0 = L[2 * (BT_TABH * sg + n)];
                            float4 E1 = L[2 * (BT_TABH * sg + n) + 1];
                            CBCT_DEV_ASSERT(__float_as_int(E1.z) - hdr.y >= 0 && __float_as_int(E1.z) - hdr.y < hdr.w);
                            E1.z = __int_as_float((int)(col0 + __float_as_int(E1.z) * (Q.XB * 16)));
                            if (sg == 0) bt_visit<0, NSLOT, TP, ZV>(acc[0], C, zlo, E0, E1, hdr.z);
                            else if (sg == 1) bt_visit<1, NSLOT, TP, ZV>(acc[0], C, zlo, E0, E1, hdr.z);
                            else if (sg == 2) bt_visit<2, NSLOT, TP, ZV>(acc[0], C, zlo, E0, E1, hdr.z);
                            else bt_visit<3, NSLOT, TP, ZV>(acc[0], C, zlo, E0, E1, hdr.z);
                        }
                    }
                    __syncwarp();
                    if (lane == 0) mbar_arrive(bar0 + 8 * (BT_NST + slot));
                }
            }
            asm volatile("cp.async.wait_group 0;" ::: "memory");
        } else {
        for (int a = 0; a < P.nbase; ++a) {
            const float4 vw = s_view[a];
#pragma unroll
            for (int rd = 0; rd < CPW; ++rd) {
                // ---- list round: every lane takes one (stage, column, candidate detector column) ----
                bool ok = false;
                float4 e0 = make_float4(0.f, 0.f, 0.f, 0.f), e1 = e0;
                if (col_ok) {
                    const int sg = rd * SPR + my_t;
                    int iu = 0;
                    ok = bt_list_entry(P, vw, rayu, a, vi0, vj0, n1, sg, cnd, e0, e1, iu);
                    if (ok) {
                        const int s_abs = 4 * a + sg, cidx = iu - s_hdr[s_abs].y;
                        CBCT_DEV_ASSERT(s_hdr[s_abs].x || (cidx >= 0 && cidx < s_hdr[s_abs].w));
                        const uint32_t col_addr = tile0 + (s_abs % BT_NST) * Q.stage_bytes + cidx * (Q.XB * 16);
                        e1.z = __int_as_float((int)col_addr);
                    }
                }
                const unsigned hit = __ballot_sync(0xffffffffu, ok);
                if (ok) {
                    const int pos = u * 8 + __popc(hit & (0xffu << (8 * u)) & lt_mask);
                    l0[pos] = e0; l1[pos] = e1;
                }
                __syncwarp();
                // ---- the round's stages ----
#pragma unroll
                for (int t = 0; t < SPR; ++t) {
                    const int sg = rd * SPR + t;
                    const int s = 4 * a + sg, slot = s % BT_NST, use = s / BT_NST;
                    mbar_wait(bar0 + 8 * slot, use & 1);
                    const int4 hdr = s_hdr[s];
                    if (!hdr.x) {
#pragma unroll
                        for (int cp = 0; cp < CPW; ++cp) {
                            const int uu = t * CPW + cp;
                            const int n_u = __popc(hit & (0xffu << (8 * uu)));
                            for (int n = 0; n < n_u; ++n) {
                                const float4 E0 = l0[uu * 8 + n], E1 = l1[uu * 8 + n];
                                if (sg == 0) bt_visit<0, NSLOT, TP, ZV>(acc[cp], C, zlo, E0, E1, hdr.z);
                                else if (sg == 1) bt_visit<1, NSLOT, TP, ZV>(acc[cp], C, zlo, E0, E1, hdr.z);
                                else if (sg == 2) bt_visit<2, NSLOT, TP, ZV>(acc[cp], C, zlo, E0, E1, hdr.z);
                                else bt_visit<3, NSLOT, TP, ZV>(acc[cp], C, zlo, E0, E1, hdr.z);
                            }
                        }
                    }
                    __syncwarp();
                    if (lane == 0) mbar_arrive(bar0 + 8 * (BT_NST + slot));
                }
            }
        }
        }
    }

    // ---------------- results: through shared memory into x-fastest order, then g = f - coef b (A4) ----------------
    __syncthreads();        // every tile has been consumed; the ring is free
    float *s_out = reinterpret_cast<float *>(smem);      // [image 8][k ZPB][rows of the image's footprint][its columns]
    if (warp < NW) {
#pragma unroll
        for (int cp = 0; cp < CPW; ++cp) {
            const int col = warp * CPW + cp, ii = col % BI, jj = col / BI;
#pragma unroll
            for (int img = 0; img < 8; ++img) {
                const int r = img & 3;
                const int wr = (r & 1) ? BJ : BI;                                  // footprint width of image r
                const int xl = r == 0 ? ii : r == 1 ? BJ - 1 - jj : r == 2 ? BI - 1 - ii : jj;
                const int yl = r == 0 ? jj : r == 1 ? ii : r == 2 ? BJ - 1 - jj : BI - 1 - ii;
#pragma unroll
                for (int v = 0; v < ZV; ++v) s_out[(img * ZPB + 32 * v + lane) * NIJ + yl * wr + xl] = acc[cp][v][img];
            }
        }
    }
    __syncthreads();
    const bool full_brick = i0 + BI <= ni && j0 + BJ <= nj;
    if (Q.vec4 && full_brick) {
        constexpr int NV4 = 8 * ZPB * NIJ / 4;
        for (int e4 = threadIdx.x; e4 < NV4; e4 += blockDim.x) {
            const int e = e4 * 4, img = e / (ZPB * NIJ), k = (e / NIJ) % ZPB, w = e % NIJ;
            const int r = img & 3, wr = (r & 1) ? BJ : BI, yl = w / wr, xl = w % wr;
            const int kk = k0 + k;
            if (kk >= Q.nzh) continue;
            const int xg = (r == 0 ? i0 : r == 1 ? P.nx - BJ - j0 : r == 2 ? P.nx - BI - i0 : j0) + xl;
            const int yg = (r == 0 ? j0 : r == 1 ? i0 : r == 2 ? P.ny - BJ - j0 : P.ny - BI - i0) + yl;
            const int zg = img >= 4 ? P.nz - 1 - kk : kk;
            const size_t o = ((size_t)zg * P.ny + yg) * P.nx + xg;
            float4 v = *reinterpret_cast<const float4 *>(s_out + e);
            if (f) {
                const float4 fv = __ldg(reinterpret_cast<const float4 *>(f + o));
                v.x = fmaf(-coef, v.x, fv.x); v.y = fmaf(-coef, v.y, fv.y); v.z = fmaf(-coef, v.z, fv.z); v.w = fmaf(-coef, v.w, fv.w);
            }
            *reinterpret_cast<float4 *>(out + o) = v;
        }
    } else {
        constexpr int NE = 8 * ZPB * NIJ;
        for (int e = threadIdx.x; e < NE; e += blockDim.x) {
            const int img = e / (ZPB * NIJ), k = (e / NIJ) % ZPB, w = e % NIJ;
            const int r = img & 3, wr = (r & 1) ? BJ : BI, yl = w / wr, xl = w % wr;
            // back to the brick's own column (ii, jj): is it inside the quadrant?
            const int ii = r == 0 ? xl : r == 1 ? yl : r == 2 ? BI - 1 - xl : BI - 1 - yl;
            const int jj = r == 0 ? yl : r == 1 ? BJ - 1 - xl : r == 2 ? BJ - 1 - yl : xl;
            const int kk = k0 + k;
            if (kk >= Q.nzh || i0 + ii >= ni || j0 + jj >= nj) continue;
            int xg, yg;
            bt_image(r, i0 + ii, j0 + jj, n1, xg, yg);
            const int zg = img >= 4 ? P.nz - 1 - kk : kk;
            const size_t o = ((size_t)zg * P.ny + yg) * P.nx + xg;
            const float v = s_out[e];
            out[o] = f ? fmaf(-coef, v, __ldg(f + o)) : v;
        }
    }
}

typedef CUresult (*EncodeTiledFn)(CUtensorMap *, CUtensorMapDataType, cuuint32_t, void *, const cuuint64_t *, const cuuint64_t *,
                                  const cuuint32_t *, const cuuint32_t *, CUtensorMapInterleave, CUtensorMapSwizzle,
                                  CUtensorMapL2promotion, CUtensorMapFloatOOBfill);

EncodeTiledFn encode_tiled_fn()
{
    static EncodeTiledFn fn = nullptr;
    if (!fn) {
        void *p = nullptr;
        cudaDriverEntryPointQueryResult qr;
        if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &p, cudaEnableDefault, &qr) == cudaSuccess &&
            qr == cudaDriverEntryPointSuccess)
            fn = reinterpret_cast<EncodeTiledFn>(p);
        else
            cudaGetLastError();
    }
    return fn;
}

template <int BI, int BJ, int CPW, int NSLOT, int TP, int MINB, int ZV, bool LT>
cbct_status bt_launch(const Level &L, const float *d_f, float coef, float *d_out, unsigned int *errflag, cudaStream_t st,
                      const Shard *sh)
{
    const LevelParams &P = L.p;
    const BtPlan &B = L.bt;
    auto kern = back_tma_kernel<BI, BJ, CPW, NSLOT, TP, MINB, ZV, LT>;
    static bool attr_set = false;       // per instantiation; the value only grows
    static int attr_bytes = 0;
    if (!attr_set || B.q.total > attr_bytes) {
        CBCT_CUDA(cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, B.q.total));
        attr_set = true; attr_bytes = B.q.total;
    }
    const int ni = P.nx / 2, nj = P.ny / 2;
    dim3 gr((ni + BI - 1) / BI, (nj + BJ - 1) / BJ, (B.q.nzh + 32 * ZV - 1) / (32 * ZV)), b((BI * BJ / CPW + 1) * 32);
    int kb_top = gr.z;
    if (sh) { kb_top = sh->zu_hi; gr.z = sh->zu_hi - sh->zu_lo; if (gr.z == 0) return CBCT_OK; }
    if (B.q.zu_fast) gr = dim3(gr.z, gr.x, gr.y);        // z-unit fastest (see the kernel)
    kern<<<gr, b, B.q.total, st>>>(B.maps, P, B.q, L.d_rayu, L.d_view, d_f, coef, d_out, errflag, kb_top, B.d_lists, B.d_hdrs);
    return CBCT_OK;
}

}  // namespace

// Plan of the TMA back-projector for one level, made once at create: which layout the residual stack takes, the tile
// sizes that hold every stage of every brick (found by walking all bricks and views in fp64, with a margin; the kernel
// counts violations in cbct_geometry::d_errflag), and the tensor maps.  plan.ok == false leaves the level to back.cu.
cbct_status bt_plan_level(const cbct_geometry *g, Level &L)
{
    const cbct_geometry_desc &d = g->desc;
    LevelParams &P = L.p;
    BtPlan &B = L.bt;
    B.ok = false;
    if (g->disable_tma || P.nsym != 4 || P.nmir != 2) return CBCT_OK;
    if (L.back_maxc > BT_MAXC) return CBCT_OK;
    // a voxel's shadow narrower than ~1.5 detector columns (in-plane voxels much finer than the pixels, config 4 and the
    // 512^3 sweep): a 4 x 4 brick then has too little work per stage for the tile ring to pay; measured 18.4 ms against
    // the list kernel's 16.4 ms at config 4, 0.84 ms against 0.95 ms at config 3 (shadow 1.9 columns)
#ifndef BT_MIN_SHADOW
#define BT_MIN_SHADOW 1.5
#endif
#ifndef BT_MAX_TABLE_GIB
#define BT_MAX_TABLE_GIB 2
#endif
    if (d.sdd / d.sad * fmin(L.hx, L.hy) / L.du < BT_MIN_SHADOW) return CBCT_OK;
    EncodeTiledFn enc = encode_tiled_fn();
    if (!enc) return CBCT_OK;
    const int BI = 4, BJ = 4;
    const int ni = P.nx / 2, nj = P.ny / 2, nzh = P.nz / 2;
    const double K = L.hz * d.sdd / L.dv;                               // K / depth = detector rows per z-index
    const double u0 = -0.5 * (P.nu - 1) * L.du + d.det_off_u;
    const double c0v_m = -(-0.5 * (P.nv - 1) * L.dv + d.det_off_v) / L.dv - 2.0e-3;
    // the first-quadrant bricks under every view = their four images under the base views
    double len_max = 0.0;
    int span_max[2] = {0, 0}, ncols_max = 0;            // row span of a block of 32 / 64 slices
    for (int a = 0; a < P.np; ++a) {
        const double c = cos(g->angles[a]), s = sin(g->angles[a]);
        const double dn = 1.01 * 0.5 * (fabs(c) * L.hx + fabs(s) * L.hy), du = 1.003 * 0.5 * (fabs(s) * L.hx + fabs(c) * L.hy);
        for (int bj = 0; bj < nj; bj += BJ)
            for (int bi = 0; bi < ni; bi += BI) {
                double lo = 1e300, hi = -1e300, rn_lo = 1e300, rn_hi = -1e300;
                for (int cj = 0; cj < 2; ++cj)
                    for (int ci = 0; ci < 2; ++ci) {
                        const int i = ci ? (bi + BI - 1 < ni ? bi + BI - 1 : ni - 1) : bi, j = cj ? (bj + BJ - 1 < nj ? bj + BJ - 1 : nj - 1) : bj;
                        const double xc = (i - 0.5 * (P.nx - 1)) * L.hx, yc = (j - 0.5 * (P.ny - 1)) * L.hy;
                        const double rn = xc * c + yc * s + d.sad, ru = xc * s - yc * c;
                        const double mag = d.sdd / rn, uc = mag * ru, W = mag * (fabs(ru / rn) * dn + du);
                        lo = fmin(lo, uc - W); hi = fmax(hi, uc + W);
                        rn_lo = fmin(rn_lo, rn); rn_hi = fmax(rn_hi, rn);
                    }
                int iu_lo = (int)ceil((lo - u0) / L.du - 0.02), iu_hi = (int)floor((hi - u0) / L.du + 0.02);
                if (iu_lo < 0) iu_lo = 0;
                if (iu_hi > P.nu - 1) iu_hi = P.nu - 1;
                if (iu_hi - iu_lo + 1 > ncols_max) ncols_max = iu_hi - iu_lo + 1;
                // rows of one voxel (lowest slice, nearest depth of the brick) and of the brick's lowest 32 slices
                const double len = K * ((double)nzh / (rn_lo - dn) - (double)(nzh - 1) / (rn_lo + dn)) + 5.0e-3;
                if (len > len_max) len_max = len;
                const double rfirst = ceil(-(double)nzh * K / (rn_lo - dn) + c0v_m) - 1.0;
                for (int zv = 1; zv <= 2; ++zv) {
                    const int klast = nzh < 32 * zv ? nzh - 1 : 32 * zv - 1;
                    const double rlast = ceil(-(double)(nzh - klast) * K / (rn_hi + dn) + c0v_m);
                    if ((int)(rlast - rfirst) > span_max[zv - 1]) span_max[zv - 1] = (int)(rlast - rfirst);
                }
            }
    }
    const int nslot = (int)floor(len_max) + 1;
    if (nslot > 4) return CBCT_OK;
    const int NSLOT = nslot <= 2 ? 2 : nslot;
    const int TP = (K / d.sad >= 1.5 && P.nv % 2 == 0) ? 2 : 1;
    const int ncols = ncols_max + 1;
    if (ncols >= (1 << BT_NMAPS)) return CBCT_OK;
    // Voxels per lane along z.  Two (blocks of 64 slices: the lists, headers and handshakes of a block serve twice the voxels, but
    // 96 registers and a doubled tile window: one block per SM) measured 0.888 ms against 0.831 ms at config 3, parity green:
    // the 17 resident warps hide less latency than the halved overhead saves.  One is the default; -DBT_ZV_MAX=2 builds the other.
#ifndef BT_ZV_MAX
#define BT_ZV_MAX 1
#endif
    BtParams &q = B.q;
    int ZV = 0, XB = 0;
    for (int zv = (nzh >= 64 ? BT_ZV_MAX : 1); zv >= 1 && !ZV; --zv) {
        // window: rows rfirst .. rlast + NSLOT, one row of alignment, the odd plane's shift, and a row of margin at each end
        const int rows = span_max[zv - 1] + NSLOT + 1 + 1 + (TP == 2 ? 3 : 1) + 2;
        XB = ((rows + TP - 1) / TP + 7) / 8 * 8;
        if (2 * XB > 256) continue;
        q.XB = XB; q.ncols = ncols; q.nzh = nzh;
        q.plane_bytes = ncols * XB * 16;
        q.half_bytes = TP * q.plane_bytes;
        q.stage_bytes = 2 * q.half_bytes;
        const int nw = BI * BJ;
        int off = BT_NST * q.stage_bytes;
        const int out_bytes = 8 * 32 * zv * BI * BJ * 4;
        if (off < out_bytes) off = out_bytes;
        q.list_off = off; off += nw * 64 * 16;
        q.view_off = off; off += P.nbase * 16;
        q.hdr_off = off; off += 4 * P.nbase * 16;
        q.bar_off = off; off += 2 * BT_NST * 8;
        q.total = off;
        if (q.total <= 227 * 1024) ZV = zv;
    }
    if (!ZV) return CBCT_OK;
    q.zu_fast = (L.nray * sizeof(float) <= ((size_t)64 << 20)) ? 1 : 0;     // the residual stack stays in L2 beside the lists
    q.ic_scale = (float)K;
    q.c0v_m = (float)c0v_m;
    q.vec4 = (P.nx % 4 == 0 && BI % 4 == 0 && BJ % 4 == 0) ? 1 : 0;
    B.BI = BI; B.BJ = BJ; B.CPW = 1; B.NSLOT = NSLOT; B.TP = TP; B.ZV = ZV;
    B.minb = (ZV == 1 && 2 * (q.total + 1024) <= 228 * 1024) ? 2 : 1;

    // the residual stack as a 4-d tensor of 8-byte elements: (2 x entry index within a plane, plane, column, base view)
    const int tXP = P.nv / TP;
    for (int b = 0; b < BT_NMAPS; ++b) {
        cuuint64_t dims[4] = {(cuuint64_t)2 * tXP, (cuuint64_t)TP, (cuuint64_t)P.nu, (cuuint64_t)P.nbase};
        cuuint64_t strides[3] = {(cuuint64_t)tXP * 16, (cuuint64_t)P.nv * 16, (cuuint64_t)P.nu * P.nv * 16};
        cuuint32_t box[4] = {(cuuint32_t)2 * XB, 1u, 1u << b, 1u};
        cuuint32_t estr[4] = {1u, 1u, 1u, 1u};
        CUresult r = enc(&B.maps.m[b], CU_TENSOR_MAP_DATA_TYPE_UINT64, 4, L.d_T, dims, strides, box, estr,
                         CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_NONE, CU_TENSOR_MAP_L2_PROMOTION_L2_256B,
                         CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
        if (r != CUDA_SUCCESS) return cbct_fail(CBCT_ERR_CUDA, "cuTensorMapEncodeTiled failed (%d)", (int)r);
    }
    P.tP = TP; P.tXP = tXP;
    B.ok = true;

    // The in-plane lists of every (first-quadrant voxel column, base view), once per geometry: 512 bytes each (84 MB at config
    // 3's finest level).  Left out -- the kernel then works its lists out itself, as in the first half of round 2 -- when an
    // image has more than BT_TABH hitting columns somewhere, when the table would pass 2 GB, or on request.
    B.d_lists = nullptr;
    const size_t n_lists = (size_t)ni * nj * P.nbase, bytes = n_lists * 512;
    if (ZV == 1 && !g->back_lists_on_the_fly && bytes <= ((size_t)BT_MAX_TABLE_GIB << 30)) {
        float4 *tab = nullptr;
        unsigned int *ovf = nullptr;
        if (cudaMalloc((void **)&tab, bytes) != cudaSuccess || cudaMalloc((void **)&ovf, sizeof(unsigned int)) != cudaSuccess) {
            cudaGetLastError(); cudaFree(tab); cudaFree(ovf);
            return CBCT_OK;                                 // no room for the table: lists on the fly
        }
        unsigned int h_ovf = 1;
        cudaMemset(tab, 0, bytes); cudaMemset(ovf, 0, sizeof(unsigned int));
        const unsigned blocks = (unsigned)((n_lists + 7) / 8);
        bt_build_lists_kernel<<<blocks, 256>>>(P, L.d_rayu, L.d_view, tab, ovf);
        const cudaError_t e = cudaMemcpy(&h_ovf, ovf, sizeof(unsigned int), cudaMemcpyDeviceToHost);
        cudaFree(ovf);
        if (e != cudaSuccess) { cudaFree(tab); return cbct_fail(CBCT_ERR_CUDA, "bt_build_lists_kernel: %s", cudaGetErrorString(e)); }
        if (h_ovf == 0) B.d_lists = tab; else cudaFree(tab);
    }
    // ... and the stage headers of every (brick, z-unit), 16 bytes per stage, with the lists
    B.d_hdrs = nullptr;
    if (B.d_lists) {
        const int gx = (ni + BI - 1) / BI, gy = (nj + BJ - 1) / BJ, gz = (nzh + 31) / 32;
        const size_t n_hdr = (size_t)gx * gy * gz * 4 * P.nbase;
        int4 *tab = nullptr;
        if (cudaMalloc((void **)&tab, n_hdr * sizeof(int4)) != cudaSuccess) { cudaGetLastError(); return CBCT_OK; }
        const unsigned blocks = (unsigned)((n_hdr + 7) / 8);
#define BT_HDR_CASE(NS, TPV) \
        if (NSLOT == NS && TP == TPV) bt_build_headers_kernel<4, 4, NS, TPV, 1><<<blocks, 256>>>(P, q, L.d_view, gx, gy, gz, tab, g->d_errflag);
        BT_HDR_CASE(2, 1) BT_HDR_CASE(3, 1) BT_HDR_CASE(4, 1) BT_HDR_CASE(2, 2) BT_HDR_CASE(3, 2) BT_HDR_CASE(4, 2)
#undef BT_HDR_CASE
        if (cudaDeviceSynchronize() != cudaSuccess) { cudaFree(tab); return cbct_fail(CBCT_ERR_CUDA, "bt_build_headers_kernel failed"); }
        B.d_hdrs = tab;
    }
    return CBCT_OK;
}

cbct_status launch_back_tma(const cbct_geometry *g, const Level &L, const float *d_f, float coef, float *d_out, cudaStream_t st,
                            const Shard *sh)
{
    const BtPlan &B = L.bt;
    cbct_status s = CBCT_ERR_INVALID_ARG;
#define BT_CASE(NS, TPV)                                                                                         \
    if (B.NSLOT == NS && B.TP == TPV) {                                                                          \
        if (B.ZV == 2) s = bt_launch<4, 4, 1, NS, TPV, 1, 2, false>(L, d_f, coef, d_out, g->d_errflag, st, sh);   \
        else if (B.d_lists && B.minb == 2) s = bt_launch<4, 4, 1, NS, TPV, 2, 1, true>(L, d_f, coef, d_out, g->d_errflag, st, sh); \
        else if (B.d_lists) s = bt_launch<4, 4, 1, NS, TPV, 1, 1, true>(L, d_f, coef, d_out, g->d_errflag, st, sh); \
        else if (B.minb == 2) s = bt_launch<4, 4, 1, NS, TPV, 2, 1, false>(L, d_f, coef, d_out, g->d_errflag, st, sh); \
        else s = bt_launch<4, 4, 1, NS, TPV, 1, 1, false>(L, d_f, coef, d_out, g->d_errflag, st, sh);             \
    }
    BT_CASE(2, 1) BT_CASE(3, 1) BT_CASE(4, 1) BT_CASE(2, 2) BT_CASE(3, 2) BT_CASE(4, 2)
#undef BT_CASE
    if (s != CBCT_OK) return s == CBCT_ERR_INVALID_ARG ? cbct_fail(s, "launch_back_tma: no kernel for this plan") : s;
    CBCT_LAUNCH_CHECK(g);
    return CBCT_OK;
}
