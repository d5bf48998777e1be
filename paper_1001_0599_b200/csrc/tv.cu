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
#include <cooperative_groups.h>
#include "cbct_internal.cuh"
#include "reduce.cuh"

namespace cg = cooperative_groups;

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

// value of the field  u = f - lam*dir  (TRIAL) or u = f  at p[o]
template <bool TRIAL>
__device__ __forceinline__ float field(const float *__restrict__ f, const float *__restrict__ dir, float lam, size_t o)
{
    return TRIAL ? fmaf(-lam, __ldg(dir + o), __ldg(f + o)) : __ldg(f + o);
}

__device__ __forceinline__ float rsqrt_ftz(float x)
{
    float r;
    asm("rsqrt.approx.ftz.f32 %0, %1;" : "=f"(r) : "f"(x));
    return r;
}

// |grad u|_delta = n2 * rsqrt(n2) (n2 >= delta^2 > 0, or exactly 0 on a flat field with delta = 0);
// inv = 1/|grad u|_delta for p = grad u * inv.
__device__ __forceinline__ float grad_norm(float gx, float gy, float gz, float delta2, float &inv)
{
    const float n2 = fmaf(gx, gx, fmaf(gy, gy, fmaf(gz, gz, delta2)));
    inv = rsqrt_ftz(n2);
    return n2 > 0.0f ? n2 * inv : 0.0f;
}

// Work decomposition of both passes: a WARP owns a tile of 32 (x, the lanes) x TV_R (y, in
// registers) voxels and marches through `zc` slices, carrying u(.,.,k+1) and p_z(.,.,k-1) in
// registers, so every voxel's value and p = grad u/|grad u| are computed ONCE per pass:
//   u(i+1,j,k)   is a warp shuffle; the values lane 31 needs (column i0+32) are loaded together
//                by lanes 0..TV_R and shuffled into place,
//   u(i,j+1,k)   is the register of the next row (one extra value-only row per tile),
//   p_y(i,j-1,k) is the previous row's register (one extra row j0-1, p_y only),
//   p_x(i-1,j,k) is a warp shuffle; the TV_R values lane 0 needs (column i0-1) are computed
//                together in lanes 0..TV_R-1 and shuffled into place.
// No shared memory and no barrier inside the march.  Loads run two slices ahead of their use
// (three register stages, rotated by unrolling the march by three).  Indices are clamped into the
// grid instead of predicated: a clamped neighbour equals the voxel itself, so the boundary rule is
// one multiplier (0 or 1) per axis, and ragged tiles compute on duplicates and mask their stores
// and sums.  Energy terms: fp32 over the TV_R rows of a slice, then fp64 per thread over the
// march, then the fixed-order block / grid reduction of reduce.cuh.
constexpr int TV_R = 4, TV_WPB = 4;

struct TvTile {
    int lane, i0, j0, k0, k1, ks;
    bool hy, hx;
    float xm, bz;
    unsigned ro[TV_R + 1];   // element offsets of rows j0 .. j0+TV_R inside a slice (clamped)
    bool rv[TV_R];           // voxel (i, j0+r) exists
    float ym[TV_R];          // multiplier of the y-neighbour of row r
    unsigned hro;            // row j0-1, this lane's column (p_y only)
    unsigned lco;            // lanes <= TV_R: voxel (i0-1, j0+lane) (p_x for lanes < TV_R; lane+1 is the y-neighbour)
    float lym;
    unsigned rco;            // lanes <= TV_R: voxel (i0+32, j0-1+lane) (value only)
    size_t plane;
};

// tile (bx, by, bz) of the grid tv_grid() lays over the volume, for the warp threadIdx.y of a 32 x TV_WPB block
__device__ __forceinline__ TvTile tv_tile(const TvDims &D, int zc, int bx, int by, int bz)
{
    TvTile T;
    T.lane = threadIdx.x;
    T.i0 = bx * 32;
    const int i = T.i0 + T.lane;
    T.j0 = (by * TV_WPB + threadIdx.y) * TV_R;
    T.k0 = bz * zc;
    T.k1 = min(T.k0 + zc, D.nz);
    T.ks = T.k0 > 0 ? T.k0 - 1 : 0;
    T.hy = T.j0 > 0;
    T.hx = T.i0 > 0;
    const float bxy = D.zero_xy ? 0.0f : 1.0f;      // out-of-grid neighbour = b * own value
    T.bz = D.zero_z ? 0.0f : 1.0f;
    T.xm = (i + 1 < D.nx) ? 1.0f : bxy;
    const int ic = min(i, D.nx - 1);
#pragma unroll
    for (int r = 0; r <= TV_R; ++r) T.ro[r] = (unsigned)(min(T.j0 + r, D.ny - 1) * D.nx + ic);
#pragma unroll
    for (int r = 0; r < TV_R; ++r) {
        T.rv[r] = i < D.nx && T.j0 + r < D.ny;
        T.ym[r] = (T.j0 + r + 1 < D.ny) ? 1.0f : bxy;
    }
    T.hro = (unsigned)(min(max(T.j0 - 1, 0), D.ny - 1) * D.nx + ic);
    const int lj = T.j0 + min(T.lane, TV_R);
    T.lco = (unsigned)(min(lj, D.ny - 1) * D.nx + max(T.i0 - 1, 0));
    T.lym = (lj + 1 < D.ny) ? 1.0f : bxy;
    const int rj = min(max(T.j0 - 1 + min(T.lane, TV_R), 0), D.ny - 1);
    T.rco = (unsigned)(rj * D.nx + min(T.i0 + 32, D.nx - 1));
    T.plane = (size_t)D.nx * D.ny;
    return T;
}

// u(i+1, row) for every lane: the next lane's value, lane 31 takes the right-column value held by
// lane `src` (a clamped duplicate of its own value at the grid's edge)
__device__ __forceinline__ float right_neighbour(float own, float rcol, int src, int lane)
{
    const float v = __shfl_down_sync(0xffffffffu, own, 1);
    const float e = __shfl_sync(0xffffffffu, rcol, src);
    return lane == 31 ? e : v;
}

// Gradient pass at u = f:  d = -div p + beta (f - g);  out[0] = sum |grad f|_delta,
// out[1] = sum (f-g)^2, out[2] = sum d^2.  FIRST: f is g itself (first descent step): no g loads.
template <bool FIRST>
__device__ __forceinline__ void tv_grad_tile(const TvDims &D, const TvTile &T, const float *__restrict__ f,
                                             const float *__restrict__ g, float beta, float delta2,
                                             float *__restrict__ d_out, double &e_tv, double &e_q, double &e_d)
{
    const float *pk = f + T.ks * T.plane;                                    // slice k
    const float *p2 = f + min(T.ks + 1, D.nz - 1) * T.plane;                 // slice k+2 (after the first advance)
    const float *pg = g + min(T.ks + 1, D.nz - 1) * T.plane;
    float *pd = d_out + T.ks * T.plane;
    // three stages: slice k, k+1, k+2
    float A[TV_R + 1], B[TV_R + 1], C[TV_R + 1], GA[TV_R], GB[TV_R], GC[TV_R];
    float hA, hB, hC = 0.0f, lA, lB, lC = 0.0f, rA, rB, rC = 0.0f;
    float pzp[TV_R];
#pragma unroll
    for (int r = 0; r <= TV_R; ++r) { A[r] = __ldg(pk + T.ro[r]); B[r] = __ldg(p2 + T.ro[r]); C[r] = 0.0f; }
#pragma unroll
    for (int r = 0; r < TV_R; ++r) {
        GA[r] = FIRST ? 0.0f : __ldg(g + T.ks * T.plane + T.ro[r]);
        GB[r] = FIRST ? 0.0f : __ldg(pg + T.ro[r]);
        GC[r] = 0.0f;
        pzp[r] = 0.0f;
    }
    hA = __ldg(pk + T.hro); hB = __ldg(p2 + T.hro);
    lA = __ldg(pk + T.lco); lB = __ldg(p2 + T.lco);
    rA = __ldg(pk + T.rco); rB = __ldg(p2 + T.rco);

    auto step = [&](int k, float (&c)[TV_R + 1], float (&cn)[TV_R + 1], float (&cnn)[TV_R + 1], float (&gc)[TV_R],
                    float (&gnn)[TV_R], float hc, float hcn, float &hcnn, float lc, float lcn, float &lcnn, float rc,
                    float &rcnn) {
        // two slices ahead (clamped at the top of the grid: those values are never used)
        if (k + 2 < D.nz) { p2 += T.plane; pg += T.plane; }
#pragma unroll
        for (int r = 0; r <= TV_R; ++r) cnn[r] = __ldg(p2 + T.ro[r]);
        if (!FIRST) {
#pragma unroll
            for (int r = 0; r < TV_R; ++r) gnn[r] = __ldg(pg + T.ro[r]);
        }
        hcnn = __ldg(p2 + T.hro); lcnn = __ldg(p2 + T.lco); rcnn = __ldg(p2 + T.rco);
        const bool ztop = k + 1 >= D.nz;
        float px[TV_R], py[TV_R], pz[TV_R], nrm[TV_R];
#pragma unroll
        for (int r = 0; r < TV_R; ++r) {
            const float xn = right_neighbour(c[r], rc, r + 1, T.lane);
            const float zn = ztop ? T.bz * c[r] : cn[r];
            const float gx = fmaf(xn, T.xm, -c[r]) * D.ihx, gy = fmaf(c[r + 1], T.ym[r], -c[r]) * D.ihy,
                        gz = (zn - c[r]) * D.ihz;
            float inv;
            nrm[r] = grad_norm(gx, gy, gz, delta2, inv);
            px[r] = gx * inv; py[r] = gy * inv; pz[r] = gz * inv;
        }
        float hpy = 0.0f, hpx = 0.0f;
        if (T.hy) {                                      // warp-uniform: row j0-1, p_y only
            const float xn = right_neighbour(hc, rc, 0, T.lane);
            const float zn = ztop ? T.bz * hc : hcn;
            const float gx = fmaf(xn, T.xm, -hc) * D.ihx, gy = (c[0] - hc) * D.ihy, gz = (zn - hc) * D.ihz;
            float inv;
            grad_norm(gx, gy, gz, delta2, inv);
            hpy = gy * inv;
        }
        if (T.hx) {                                      // warp-uniform: column i0-1, p_x only, rows in lanes 0..TV_R-1
            // its x-neighbour is lane 0's voxel of the same row, its y-neighbour the next lane's voxel
            float xn = 0.0f;
#pragma unroll
            for (int r = 0; r < TV_R; ++r) {
                const float v = __shfl_sync(0xffffffffu, c[r], 0);
                if (T.lane == r) xn = v;
            }
            const float yn = __shfl_down_sync(0xffffffffu, lc, 1);
            const float zn = ztop ? T.bz * lc : lcn;
            const float gx = (xn - lc) * D.ihx, gy = fmaf(yn, T.lym, -lc) * D.ihy, gz = (zn - lc) * D.ihz;
            float inv;
            grad_norm(gx, gy, gz, delta2, inv);
            hpx = gx * inv;
        }
        const bool emit = k >= T.k0;                     // the slice before the chunk only supplies p_z
        float s_tv = 0.0f, s_q = 0.0f, s_d = 0.0f;
#pragma unroll
        for (int r = 0; r < TV_R; ++r) {
            float left = __shfl_up_sync(0xffffffffu, px[r], 1);
            const float edge = __shfl_sync(0xffffffffu, hpx, r);
            if (T.lane == 0) left = edge;
            const float up = r > 0 ? py[r > 0 ? r - 1 : 0] : hpy;
            const float div = (px[r] - left) * D.ihx + (py[r] - up) * D.ihy + (pz[r] - pzp[r]) * D.ihz;
            const float res = FIRST ? 0.0f : c[r] - gc[r];
            const float dd = FIRST ? -div : fmaf(beta, res, -div);
            if (emit && T.rv[r]) {
                pd[T.ro[r]] = dd;
                s_tv += nrm[r];
                if (!FIRST) s_q = fmaf(res, res, s_q);
                s_d = fmaf(dd, dd, s_d);
            }
            pzp[r] = pz[r];
        }
        e_tv += (double)s_tv; e_d += (double)s_d;
        if (!FIRST) e_q += (double)s_q;
        pk += T.plane; pd += T.plane;
    };

    for (int k = T.ks; k < T.k1; k += 3) {
        step(k, A, B, C, GA, GC, hA, hB, hC, lA, lB, lC, rA, rC);
        if (k + 1 >= T.k1) break;
        step(k + 1, B, C, A, GB, GA, hB, hC, hA, lB, lC, lA, rB, rA);
        if (k + 2 >= T.k1) break;
        step(k + 2, C, A, B, GC, GB, hC, hA, hB, lC, lA, lB, rC, rB);
    }
}

// Energy pass at u = f - lam*dir (TRIAL) or u = f:  out[0] = sum |grad u|_delta and, when rows == 2,
// out[1] = sum (u-g)^2.  Same warp tiles and march; nothing but u(i+1) is exchanged between voxels.
template <bool TRIAL>
__device__ __forceinline__ void tv_energy_tile(const TvDims &D, const TvTile &T, const float *__restrict__ f,
                                               const float *__restrict__ dir, const float *__restrict__ g, float lam,
                                               float delta2, float *__restrict__ cand, int cand_clip, double &e_tv, double &e_q)
{
    const bool hasg = g != nullptr;
    const size_t ok = T.k0 * T.plane;
    size_t ocur = ok;                                             // slice k
    size_t o2 = min(T.k0 + 1, D.nz - 1) * T.plane;                // slice k+2 (after the first advance)
    float A[TV_R + 1], B[TV_R + 1], C[TV_R + 1], GA[TV_R], GB[TV_R], GC[TV_R];
    float rA, rB, rC = 0.0f;
#pragma unroll
    for (int r = 0; r <= TV_R; ++r) {
        A[r] = field<TRIAL>(f, dir, lam, ok + T.ro[r]);
        B[r] = field<TRIAL>(f, dir, lam, o2 + T.ro[r]);
        C[r] = 0.0f;
    }
#pragma unroll
    for (int r = 0; r < TV_R; ++r) {
        GA[r] = hasg ? __ldg(g + ok + T.ro[r]) : 0.0f;
        GB[r] = hasg ? __ldg(g + o2 + T.ro[r]) : 0.0f;
        GC[r] = 0.0f;
    }
    rA = field<TRIAL>(f, dir, lam, ok + T.rco); rB = field<TRIAL>(f, dir, lam, o2 + T.rco);

    auto step = [&](int k, float (&c)[TV_R + 1], float (&cn)[TV_R + 1], float (&cnn)[TV_R + 1], float (&gc)[TV_R],
                    float (&gnn)[TV_R], float rc, float &rcnn) {
        if (k + 2 < D.nz) o2 += T.plane;
#pragma unroll
        for (int r = 0; r <= TV_R; ++r) cnn[r] = field<TRIAL>(f, dir, lam, o2 + T.ro[r]);
        if (hasg) {
#pragma unroll
            for (int r = 0; r < TV_R; ++r) gnn[r] = __ldg(g + o2 + T.ro[r]);
        }
        rcnn = field<TRIAL>(f, dir, lam, o2 + T.rco);
        const bool ztop = k + 1 >= D.nz;
        float s_tv = 0.0f, s_q = 0.0f;
#pragma unroll
        for (int r = 0; r < TV_R; ++r) {
            const float xn = right_neighbour(c[r], rc, r + 1, T.lane);
            const float zn = ztop ? T.bz * c[r] : cn[r];
            const float gx = fmaf(xn, T.xm, -c[r]) * D.ihx, gy = fmaf(c[r + 1], T.ym[r], -c[r]) * D.ihy,
                        gz = (zn - c[r]) * D.ihz;
            float inv;
            const float nrm = grad_norm(gx, gy, gz, delta2, inv);
            const float res = c[r] - gc[r];
            if (T.rv[r]) {
                s_tv += nrm; s_q = fmaf(res, res, s_q);
                // the trial volume itself, truncated as the LAST update would: if the step is accepted and is the last
                // one, this is the result and the update pass is skipped (same expression as tv_update_kernel)
                if (TRIAL && cand) cand[ocur + T.ro[r]] = (cand_clip && c[r] < 0.0f) ? 0.0f : c[r];
            }
        }
        e_tv += (double)s_tv; e_q += (double)s_q;
        ocur += T.plane;
    };

    for (int k = T.k0; k < T.k1; k += 3) {
        step(k, A, B, C, GA, GC, rA, rC);
        if (k + 1 >= T.k1) break;
        step(k + 1, B, C, A, GB, GA, rB, rA);
        if (k + 2 >= T.k1) break;
        step(k + 2, C, A, B, GC, GB, rC, rB);
    }
}

// ---------------------------------------------------------------------------------------------------------------------
// The 16-byte form of the warp tiles (volumes with nx % 4 == 0, nx >= 128 and 16-byte aligned rows): a lane owns FOUR
// consecutive voxels of a row, so a warp tile is 128 (x) x TQ_R (y) voxels and every access is a 16-byte load or store of
// a whole 128-byte line per quarter warp.  Same stencil, same boundary rules and the same per-voxel fp32 expressions as the
// tiles above; what changes is the bookkeeping per voxel: one shuffle pair per FOUR voxels for u(i+1) and p_x(i-1), a
// quarter of the load / store instructions, and the row j0-1 that supplies p_y(.,j0-1) is a register row like the others.
// Loads run one to two slices ahead WITHOUT extra buffers: a row of slice k is dead once its own row and the row below it
// are done, and is refilled with the same row of slice k+2 on the spot (the march is unrolled by two, the two register
// sets swapping roles), so every load has a whole slice of arithmetic to land.
// ---------------------------------------------------------------------------------------------------------------------
constexpr int TQ_R = 4;       // rows per warp tile
constexpr int TQ_V = 4;       // consecutive voxels per lane: 16-byte accesses (2, with 8-byte accesses, measured 25-30 % slower)
constexpr int TQ_W = 32 * TQ_V;   // voxels per warp tile row

struct F4 { float v[TQ_V]; };
// Streaming loads: read-only path, no L1 line allocated -- the gradient pass's rings leave the SM ~20 KB of L1, and every
// line a streaming load allocates there is one fewer load in flight.
__device__ __forceinline__ F4 ldg4(const float *__restrict__ p)
{
    F4 r;
    asm volatile("ld.global.nc.L1::no_allocate.v4.f32 {%0, %1, %2, %3}, [%4];" : "=f"(r.v[0]), "=f"(r.v[1]), "=f"(r.v[2]), "=f"(r.v[3]) : "l"(p) : "memory");
    return r;
}
__device__ __forceinline__ float ldg1(const float *__restrict__ p)
{
    float r;
    asm volatile("ld.global.nc.L1::no_allocate.f32 %0, [%1];" : "=f"(r) : "l"(p) : "memory");
    return r;
}
__device__ __forceinline__ void st4(float *__restrict__ p, const F4 &a)
{
    asm volatile("st.global.v4.f32 [%0], {%1, %2, %3, %4};" ::"l"(p), "f"(a.v[0]), "f"(a.v[1]), "f"(a.v[2]), "f"(a.v[3]) : "memory");
}

struct TqTile {
    int lane, k0, k1, ks;
    bool hy, hx, xedge;        // row j0-1 / column i0-1 exists; the lane's last voxel is the last of its row
    float xm, bz;
    unsigned ro[TQ_R + 2];     // element offsets inside a slice of rows j0-1 .. j0+TQ_R (clamped), at the lane's first voxel
    bool rv[TQ_R];             // voxels (i..i+3, j0+r) exist
    float ym[TQ_R + 1];        // multiplier of the y-neighbour of rows j0-1 .. j0+TQ_R-1
    unsigned lco;              // lanes <= TQ_R: voxel (i0-1, j0+lane)        (p_x of the column left of the tile)
    float lym;
    unsigned rco;              // lanes <= TQ_R: voxel (i0+128, j0-1+lane)    (u(i+1) of lane 31)
    size_t plane;
};

// `ntz` = number of z-chunks: chunk bz holds slices [bz nz / ntz, (bz+1) nz / ntz) -- balanced, so that the host can fit the
// tile count to the blocks resident at once (tv_tiling)
__device__ __forceinline__ TqTile tq_tile(const TvDims &D, int ntz, int bx, int by, int bz)
{
    TqTile T;
    T.lane = threadIdx.x;
    const int i0 = bx * TQ_W, i = i0 + TQ_V * T.lane;
    const int j0 = (by * TV_WPB + threadIdx.y) * TQ_R;
    T.k0 = (int)(((long long)bz * D.nz) / ntz);
    T.k1 = (int)(((long long)(bz + 1) * D.nz) / ntz);
    T.ks = T.k0 > 0 ? T.k0 - 1 : 0;
    T.hy = j0 > 0;
    T.hx = i0 > 0;
    const float bxy = D.zero_xy ? 0.0f : 1.0f;
    T.bz = D.zero_z ? 0.0f : 1.0f;
    T.xedge = i + TQ_V >= D.nx;
    T.xm = T.xedge ? bxy : 1.0f;
    const int ic = min(i, D.nx - TQ_V);
#pragma unroll
    for (int q = 0; q <= TQ_R + 1; ++q) T.ro[q] = (unsigned)(min(max(j0 - 1 + q, 0), D.ny - 1) * D.nx + ic);
#pragma unroll
    for (int r = 0; r < TQ_R; ++r) T.rv[r] = i < D.nx && j0 + r < D.ny;
#pragma unroll
    for (int q = 0; q <= TQ_R; ++q) T.ym[q] = (j0 + q < D.ny) ? 1.0f : bxy;        // row j0-1+q, neighbour j0+q
    const int lj = j0 + min(T.lane, TQ_R);
    T.lco = (unsigned)(min(lj, D.ny - 1) * D.nx + max(i0 - 1, 0));
    T.lym = (lj + 1 < D.ny) ? 1.0f : bxy;
    const int rj = min(max(j0 - 1 + min(T.lane, TQ_R), 0), D.ny - 1);
    T.rco = (unsigned)(rj * D.nx + min(i0 + TQ_W, D.nx - 1));
    T.plane = (size_t)D.nx * D.ny;
    return T;
}

// forward differences of the four voxels of a lane: c = u(i..i+3, j, k), yv = u(., j+1, k), zn = u(., ., k+1) (already the
// boundary value at the top of the grid), xr = u(i+4, j, k)
__device__ __forceinline__ void tq_gradient(const TvDims &D, const F4 &c, const F4 &yv, const F4 &zn, float xr, float xm, float ym,
                                            float delta2, F4 &gx, F4 &gy, F4 &gz, F4 &inv, F4 &nrm)
{
#pragma unroll
    for (int e = 0; e + 1 < TQ_V; ++e) gx.v[e] = (c.v[e + 1] - c.v[e]) * D.ihx;
    gx.v[TQ_V - 1] = fmaf(xr, xm, -c.v[TQ_V - 1]) * D.ihx;
#pragma unroll
    for (int e = 0; e < TQ_V; ++e) {
        gy.v[e] = fmaf(yv.v[e], ym, -c.v[e]) * D.ihy;
        gz.v[e] = (zn.v[e] - c.v[e]) * D.ihz;
        nrm.v[e] = grad_norm(gx.v[e], gy.v[e], gz.v[e], delta2, inv.v[e]);
    }
}

// The gradient pass with its loads staged through shared memory by cp.async (sm_80+ LDGSTS; 16 bytes per lane, L1 bypassed):
// every warp owns a ring of three slices x (R+2) rows of u and two slices x R rows of g, 13 KB, filled two slices ahead of
// the arithmetic by the lanes that will read it (no block barrier: a lane reads back its own 16 bytes; the one cross-lane read
// -- lane 0's first voxel for the column left of the tile -- follows a __syncwarp).  The slices in flight cost no registers,
// so the pass keeps 16 warps per SM where the register-staged form above spilled under the 128-register cap of the
// cooperative kernel.  Same arithmetic, same order of operations per voxel, same sums.
constexpr int TQ_RING = 3;
constexpr int TQ_SMEM_PER_WARP = (TQ_RING * (TQ_R + 2) + 2 * TQ_R) * 32 * 16;      // bytes
constexpr int TQ_SMEM_PER_BLOCK = TQ_SMEM_PER_WARP * TV_WPB;

__device__ __forceinline__ void cp_async16(uint32_t dst, const float *src)
{
    asm volatile("cp.async.cg.shared.global [%0], [%1], 16;" ::"r"(dst), "l"(src) : "memory");
}
__device__ __forceinline__ void cp_async_commit() { asm volatile("cp.async.commit_group;" ::: "memory"); }
template <int N> __device__ __forceinline__ void cp_async_wait() { asm volatile("cp.async.wait_group %0;" ::"n"(N) : "memory"); }
__device__ __forceinline__ F4 lds4(uint32_t a)
{
    F4 r;
    asm volatile("ld.shared.v4.f32 {%0, %1, %2, %3}, [%4];" : "=f"(r.v[0]), "=f"(r.v[1]), "=f"(r.v[2]), "=f"(r.v[3]) : "r"(a) : "memory");
    return r;
}
__device__ __forceinline__ float lds1(uint32_t a)
{
    float r;
    asm volatile("ld.shared.f32 %0, [%1];" : "=f"(r) : "r"(a) : "memory");
    return r;
}

// this warp's ring in the block's dynamic shared memory (TQ_SMEM_PER_BLOCK bytes)
extern __shared__ __align__(16) unsigned char tq_dyn_smem[];
__device__ __forceinline__ uint32_t tq_ring_base()
{
    return (uint32_t)__cvta_generic_to_shared(tq_dyn_smem) + threadIdx.y * TQ_SMEM_PER_WARP;
}

template <bool FIRST>
__device__ __forceinline__ void tq_grad_tile_async(const TvDims &D, const TqTile &T, const float *__restrict__ f,
                                                   const float *__restrict__ g, float beta, float delta2,
                                                   float *__restrict__ d_out, uint32_t ring, double &e_tv, double &e_q, double &e_d)
{
    static_assert(TQ_V == 4, "cp.async stages 16 bytes per lane");
    constexpr int R = TQ_R;
    const size_t pl = T.plane;
    const int ztopk = D.nz - 1, kend = min(T.k1, ztopk);
    // ring addresses of this lane: slice s, row q -> ring + ((s % 3) * (R+2) + q) * 512 + lane * 16; g: gring + ((s & 1) * R + r) * 512
    const uint32_t fr = ring + T.lane * 16, gr = ring + TQ_RING * (R + 2) * 512 + T.lane * 16;
    auto issue_f = [&](int slice, int slot) {
        const float *ps = f + (size_t)slice * pl;
#pragma unroll
        for (int q = 0; q <= R + 1; ++q) cp_async16(fr + (slot * (R + 2) + q) * 512, ps + T.ro[q]);
    };
    auto issue_g = [&](int slice, int slot) {
        if (FIRST) return;
        const float *ps = g + (size_t)slice * pl;
#pragma unroll
        for (int r = 0; r < R; ++r) cp_async16(gr + (slot * R + r) * 512, ps + T.ro[r + 1]);
    };
    F4 pzp[R];
#pragma unroll
    for (int r = 0; r < R; ++r)
#pragma unroll
        for (int e = 0; e < TQ_V; ++e) pzp[r].v[e] = 0.0f;
    int s0 = T.ks % TQ_RING;                              // ring slot of slice k
    issue_f(T.ks, s0); issue_g(T.ks, T.ks & 1); cp_async_commit();
    issue_f(min(T.ks + 1, ztopk), (s0 + 1) % TQ_RING); cp_async_commit();
    float lc = ldg1(f + (size_t)T.ks * pl + T.lco), ln = ldg1(f + (size_t)min(T.ks + 1, ztopk) * pl + T.lco);
    float rc = ldg1(f + (size_t)T.ks * pl + T.rco), rn = ldg1(f + (size_t)min(T.ks + 1, ztopk) * pl + T.rco);

    for (int k = T.ks; k < T.k1; ++k) {
        const int s1 = s0 + 1 == TQ_RING ? 0 : s0 + 1, s2 = s1 + 1 == TQ_RING ? 0 : s1 + 1;
        issue_f(min(k + 2, kend), s2); issue_g(min(k + 1, T.k1 - 1), (k + 1) & 1); cp_async_commit();
        const float l2 = ldg1(f + (size_t)min(k + 2, kend) * pl + T.lco), r2 = ldg1(f + (size_t)min(k + 2, kend) * pl + T.rco);
        cp_async_wait<1>();                              // slices k, k+1 and g(k) have landed
        __syncwarp();
        float *pd = d_out + (size_t)k * pl;
        const bool ztop = k + 1 >= D.nz, emit = k >= T.k0;
        const uint32_t fc = fr + s0 * (R + 2) * 512, fn = fr + s1 * (R + 2) * 512, gc = gr + (k & 1) * R * 512;
        if (ztop) ln = T.bz * lc;
        float hpx = 0.0f;
        if (T.hx) {                                      // warp-uniform: column i0-1, p_x only, its rows in lanes 0..R-1
            const float xn = lds1(fc - T.lane * 16 + (min(T.lane, R - 1) + 1) * 512);     // lane 0's first voxel of row j0+lane
            const float yn = __shfl_down_sync(0xffffffffu, lc, 1);
            const float gx = (xn - lc) * D.ihx, gy = fmaf(yn, T.lym, -lc) * D.ihy, gz = (ln - lc) * D.ihz;
            float inv;
            grad_norm(gx, gy, gz, delta2, inv);
            hpx = gx * inv;
        }
        F4 pyp, cq = lds4(fc);
#pragma unroll
        for (int e = 0; e < TQ_V; ++e) pyp.v[e] = 0.0f;
        float s_tv = 0.0f, s_q = 0.0f, s_d = 0.0f;
#pragma unroll
        for (int q = 0; q <= R; ++q) {                   // rows j0-1 (p_y only) .. j0+R-1
            const F4 cy = lds4(fc + (q + 1) * 512);
            if (q > 0 || T.hy) {
                F4 zn, gx, gy, gz, inv, nrm;
                if (ztop) {
#pragma unroll
                    for (int e = 0; e < TQ_V; ++e) zn.v[e] = T.bz * cq.v[e];
                } else {
                    zn = lds4(fn + q * 512);
                }
                float xr = __shfl_down_sync(0xffffffffu, cq.v[0], 1);
                const float ed = __shfl_sync(0xffffffffu, rc, q);
                if (T.lane == 31) xr = ed;
                if (T.xedge) xr = cq.v[TQ_V - 1];
                tq_gradient(D, cq, cy, zn, xr, T.xm, T.ym[q], delta2, gx, gy, gz, inv, nrm);
                if (q == 0) {
#pragma unroll
                    for (int e = 0; e < TQ_V; ++e) pyp.v[e] = gy.v[e] * inv.v[e];
                } else {
                    const int r = q - 1;
                    F4 px, dd, G;
                    if (!FIRST) G = lds4(gc + r * 512);
#pragma unroll
                    for (int e = 0; e < TQ_V; ++e) px.v[e] = gx.v[e] * inv.v[e];
                    float left = __shfl_up_sync(0xffffffffu, px.v[TQ_V - 1], 1);
                    const float edge = __shfl_sync(0xffffffffu, hpx, r);
                    if (T.lane == 0) left = edge;
#pragma unroll
                    for (int e = 0; e < TQ_V; ++e) {
                        const float py = gy.v[e] * inv.v[e], pz = gz.v[e] * inv.v[e];
                        const float div = (px.v[e] - (e == 0 ? left : px.v[e > 0 ? e - 1 : 0])) * D.ihx + (py - pyp.v[e]) * D.ihy +
                                          (pz - pzp[r].v[e]) * D.ihz;
                        const float res = FIRST ? 0.0f : cq.v[e] - G.v[e];
                        dd.v[e] = FIRST ? -div : fmaf(beta, res, -div);
                        pyp.v[e] = py; pzp[r].v[e] = pz;
                        if (emit && T.rv[r]) {
                            s_tv += nrm.v[e];
                            if (!FIRST) s_q = fmaf(res, res, s_q);
                            s_d = fmaf(dd.v[e], dd.v[e], s_d);
                        }
                    }
                    if (emit && T.rv[r]) st4(pd + T.ro[q], dd);
                }
            }
            cq = cy;
        }
        e_tv += (double)s_tv; e_d += (double)s_d;
        if (!FIRST) e_q += (double)s_q;
        lc = ln; ln = l2; rc = rn; rn = r2;
        s0 = s1;
    }
    cp_async_wait<0>();
}

// Energy pass on the 16-byte tiles: rows j0 .. j0+R-1 and the value-only row j0+R.  TRIAL: u = f - lam dir, combined one slice
// after its two loads were issued (the raw f sits in the register row that will hold u, the raw dir in `rawd`).
template <bool TRIAL>
__device__ __forceinline__ void tq_energy_tile(const TvDims &D, const TqTile &T, const float *__restrict__ f,
                                               const float *__restrict__ dir, const float *__restrict__ g, float lam,
                                               float delta2, float *__restrict__ cand, int cand_clip, double &e_tv, double &e_q)
{
    constexpr int R = TQ_R;
    const bool hasg = g != nullptr;
    const size_t pl = T.plane;
    const int ztopk = D.nz - 1, kend = min(T.k1, ztopk);
    F4 A[R + 1], B[R + 1], rawd[R + 1], G[R];
    float rA, rB, rD = 0.0f;
    const unsigned *ro = T.ro + 1;                                        // rows j0 .. j0+R
    const unsigned rco = __shfl_down_sync(0xffffffffu, T.rco, 1);         // lanes <= R: voxel (i0+128, j0+lane)
    {
        const size_t o0 = (size_t)T.k0 * pl, o1 = (size_t)min(T.k0 + 1, ztopk) * pl;
#pragma unroll
        for (int q = 0; q <= R; ++q) {
            A[q] = ldg4(f + o0 + ro[q]); B[q] = ldg4(f + o1 + ro[q]);
            if (TRIAL) {
                const F4 d0 = ldg4(dir + o0 + ro[q]);
                rawd[q] = ldg4(dir + o1 + ro[q]);
#pragma unroll
                for (int e = 0; e < TQ_V; ++e) A[q].v[e] = fmaf(-lam, d0.v[e], A[q].v[e]);
            }
        }
#pragma unroll
        for (int r = 0; r < R; ++r) {
            if (hasg) G[r] = ldg4(g + o0 + ro[r]);
            else {
#pragma unroll
                for (int e = 0; e < TQ_V; ++e) G[r].v[e] = 0.0f;
            }
        }
        rA = ldg1(f + o0 + rco); rB = ldg1(f + o1 + rco);
        if (TRIAL) { rA = fmaf(-lam, ldg1(dir + o0 + rco), rA); rD = ldg1(dir + o1 + rco); }
    }

    auto step = [&](int k, F4 (&c)[R + 1], F4 (&n)[R + 1], float &rc, float &rn) {
        const size_t o2 = (size_t)min(k + 2, kend) * pl, og = (size_t)min(k + 1, T.k1 - 1) * pl, ok = (size_t)k * pl;
        const bool ztop = k + 1 >= D.nz;
        if (TRIAL) {                                      // slice k+1: combine what the last step loaded
#pragma unroll
            for (int q = 0; q <= R; ++q)
#pragma unroll
                for (int e = 0; e < TQ_V; ++e) n[q].v[e] = fmaf(-lam, rawd[q].v[e], n[q].v[e]);
            rn = fmaf(-lam, rD, rn);
        }
        if (ztop) {
#pragma unroll
            for (int q = 0; q < R; ++q)
#pragma unroll
                for (int e = 0; e < TQ_V; ++e) n[q].v[e] = T.bz * c[q].v[e];
        }
        float s_tv = 0.0f, s_q = 0.0f;
#pragma unroll
        for (int q = 0; q < R; ++q) {
            F4 gx, gy, gz, inv, nrm;
            float xr = __shfl_down_sync(0xffffffffu, c[q].v[0], 1);
            const float ed = __shfl_sync(0xffffffffu, rc, q);
            if (T.lane == 31) xr = ed;
            if (T.xedge) xr = c[q].v[TQ_V - 1];
            tq_gradient(D, c[q], c[q + 1], n[q], xr, T.xm, T.ym[q + 1], delta2, gx, gy, gz, inv, nrm);
            if (T.rv[q]) {
                F4 o;
#pragma unroll
                for (int e = 0; e < TQ_V; ++e) {
                    const float res = c[q].v[e] - G[q].v[e];
                    s_tv += nrm.v[e]; s_q = fmaf(res, res, s_q);
                    o.v[e] = (cand_clip && c[q].v[e] < 0.0f) ? 0.0f : c[q].v[e];
                }
                if (TRIAL && cand) st4(cand + ok + ro[q], o);
            }
            if (hasg) G[q] = ldg4(g + og + ro[q]);
            c[q] = ldg4(f + o2 + ro[q]);
            if (TRIAL) rawd[q] = ldg4(dir + o2 + ro[q]);
        }
        c[R] = ldg4(f + o2 + ro[R]);
        if (TRIAL) rawd[R] = ldg4(dir + o2 + ro[R]);
        rc = ldg1(f + o2 + rco);
        if (TRIAL) rD = ldg1(dir + o2 + rco);
        e_tv += (double)s_tv; e_q += (double)s_q;
    };

    for (int k = T.k0; k < T.k1; k += 2) {
        step(k, A, B, rA, rB);
        if (k + 1 >= T.k1) break;
        step(k + 1, B, A, rB, rA);
    }
}

// The passes as kernels of their own (the host-sequenced loop, cbct_tv_energy): one block per tile.  VEC: the 16-byte tiles.
template <bool FIRST, bool VEC>
__global__ void __launch_bounds__(32 * TV_WPB)
tv_grad_kernel(const TvDims D, const float *__restrict__ f, const float *__restrict__ g, float beta, float delta2,
               float *__restrict__ d_out, int zc, double *__restrict__ partials, int stride,
               unsigned int *__restrict__ counter, double *__restrict__ out)
{
    __shared__ double slot[32];
    double e_tv = 0.0, e_q = 0.0, e_d = 0.0;
    if (VEC) {
        const TqTile T = tq_tile(D, zc, blockIdx.x, blockIdx.y, blockIdx.z);
        tq_grad_tile_async<FIRST>(D, T, f, g, beta, delta2, d_out, tq_ring_base(), e_tv, e_q, e_d);
    } else {
        const TvTile T = tv_tile(D, zc, blockIdx.x, blockIdx.y, blockIdx.z);
        tv_grad_tile<FIRST>(D, T, f, g, beta, delta2, d_out, e_tv, e_q, e_d);
    }
    double s[3];
    s[0] = block_sum(e_tv, slot);
    s[1] = block_sum(e_q, slot);
    s[2] = block_sum(e_d, slot);
    publish_and_finalize<3>(s, 3, partials, stride, counter, out, slot);
}

template <bool TRIAL, bool VEC>
__global__ void __launch_bounds__(32 * TV_WPB)
tv_energy_kernel(const TvDims D, const float *__restrict__ f, const float *__restrict__ dir,
                 const float *__restrict__ g, float lam, float delta2, int zc, int rows,
                 double *__restrict__ partials, int stride, unsigned int *__restrict__ counter,
                 double *__restrict__ out, float *__restrict__ cand, int cand_clip)
{
    __shared__ double slot[32];
    double e_tv = 0.0, e_q = 0.0;
    if (VEC) {
        const TqTile T = tq_tile(D, zc, blockIdx.x, blockIdx.y, blockIdx.z);
        tq_energy_tile<TRIAL>(D, T, f, dir, g, lam, delta2, cand, cand_clip, e_tv, e_q);
    } else {
        const TvTile T = tv_tile(D, zc, blockIdx.x, blockIdx.y, blockIdx.z);
        tv_energy_tile<TRIAL>(D, T, f, dir, g, lam, delta2, cand, cand_clip, e_tv, e_q);
    }
    double s[2];
    s[0] = block_sum(e_tv, slot);
    s[1] = g != nullptr ? block_sum(e_q, slot) : 0.0;
    publish_and_finalize<2>(s, rows, partials, stride, counter, out, slot);
}

// out = f - lam * d  (optionally clipped at 0: Algorithm A1 step 3, L149); d == NULL: out = f.
// Plain loads and no __restrict__: out may be f itself (each thread reads an element, then writes it).
template <typename V>
__global__ void tv_update_kernel(size_t n, const V *f, const V *d, float lam, int clip, V *out);

template <>
__global__ void tv_update_kernel<float>(size_t n, const float *f, const float *d, float lam, int clip, float *out)
{
    for (size_t o = (size_t)blockIdx.x * blockDim.x + threadIdx.x; o < n; o += (size_t)gridDim.x * blockDim.x) {
        float v = d ? fmaf(-lam, d[o], f[o]) : f[o];
        out[o] = (clip && v < 0.0f) ? 0.0f : v;
    }
}

template <>
__global__ void tv_update_kernel<float4>(size_t n, const float4 *f, const float4 *d, float lam, int clip, float4 *out)
{
    for (size_t o = (size_t)blockIdx.x * blockDim.x + threadIdx.x; o < n; o += (size_t)gridDim.x * blockDim.x) {
        float4 v = f[o];
        if (d) {
            const float4 w = d[o];
            v.x = fmaf(-lam, w.x, v.x); v.y = fmaf(-lam, w.y, v.y); v.z = fmaf(-lam, w.z, v.z); v.w = fmaf(-lam, w.w, v.w);
        }
        if (clip) {     // (v < 0) ? 0 : v, so that -0 and NaN pass through like the scalar path
            v.x = v.x < 0.0f ? 0.0f : v.x; v.y = v.y < 0.0f ? 0.0f : v.y;
            v.z = v.z < 0.0f ? 0.0f : v.z; v.w = v.w < 0.0f ? 0.0f : v.w;
        }
        out[o] = v;
    }
}

// ---------------------------------------------------------------------------------------------------------------------
// The whole TV-prox call as ONE cooperative kernel: the Armijo loop of L155-L159 runs on the device.
//
// A persistent grid (as many blocks as fit the GPU at once) walks the tiles of every pass; between passes a grid-wide
// barrier, after which EVERY block adds the blocks' fp64 partial sums in index order -- the same number in every block, so
// all blocks take the same accept / shrink / stop decision (Eq. 5; the epsilon rule) without a host round trip and
// without a second kernel.  Passes, buffers and the order of the decisions are those of the host-sequenced loop
// (run_tv_prox below): gradient pass, trial passes with lam = 1/beta, alpha/beta, ..., update, and the truncated trial
// volume doubling as the result when the accepted step is the last.  Sums depend on the grid size only (fixed for a
// device), never on timing: bitwise reproducible.
// ---------------------------------------------------------------------------------------------------------------------
// a 16-byte load that does not allocate an L1 line (plain ld: the target may be written by the same thread afterwards)
__device__ __forceinline__ float4 ld_stream4(const float4 *p)
{
    float4 v;
    asm volatile("ld.global.L1::no_allocate.v4.f32 {%0, %1, %2, %3}, [%4];" : "=f"(v.x), "=f"(v.y), "=f"(v.z), "=f"(v.w) : "l"(p) : "memory");
    return v;
}

struct TvCoop {
    TvDims D;
    const float *g;
    float *f, *f2, *d;
    double beta, armijo_c, alpha, rel_tol, n;
    float delta2;
    int max_inner, max_bt, nonneg, zc, ntx, nty, ntz;
    size_t nvox;
    double *partials;       // 6 rows of `stride` per-TILE partials (two sets of three, used in turn)
    int stride;
    unsigned int *ticket;   // two tile counters, used in turn by successive passes; 0 between calls
    double *report;         // [0] inner, [1] trials, [2] E_first, [3] E_last of this call; [4], [5] += inner, trials
};

template <bool VEC>
__global__ void __launch_bounds__(32 * TV_WPB, 4)
tv_prox_coop_kernel(const TvCoop p)
{
    cg::grid_group grid = cg::this_grid();
    __shared__ double slot[32];
    __shared__ double s_tot[3];
    const int tid = threadIdx.y * 32 + threadIdx.x, nthr = 32 * TV_WPB;
    const int ntiles = p.ntx * p.nty * p.ntz;
    const unsigned nblk = gridDim.x;
    int pset = 0;
    __shared__ int s_tile;

    // The tiles of a pass are handed out by a ticket counter (the blocks stay evenly loaded whatever ntiles / gridDim is);
    // every tile publishes its own partial sums, so which block computed a tile does not enter any sum.
    auto next_tile = [&]() {
        __syncthreads();
        if (tid == 0) s_tile = (int)atomicAdd(p.ticket + pset, 1u);
        __syncthreads();
        return s_tile;
    };
    auto publish = [&](int t, double a0, double a1, double a2, int rows) {
        const double v[3] = {a0, a1, a2};
        for (int r = 0; r < rows; ++r) {
            const double s = block_sum(v[r], slot);
            if (tid == 0) p.partials[(size_t)(pset * 3 + r) * p.stride + t] = s;
        }
    };
    // grid barrier, then every block adds all tiles' partials in tile order: the same totals in every thread of the grid
    auto grid_sums = [&](int rows, double (&tot)[3]) {
        grid.sync();
        if (blockIdx.x == 0 && tid == 0) p.ticket[pset] = 0u;        // free again two passes from now
        for (int r = 0; r < rows; ++r) {
            double acc = 0.0;
            for (int i = tid; i < ntiles; i += nthr) acc += __ldcg(p.partials + (size_t)(pset * 3 + r) * p.stride + i);
            const double s = block_sum(acc, slot);
            if (tid == 0) s_tot[r] = s;
        }
        __syncthreads();
        for (int r = 0; r < rows; ++r) tot[r] = s_tot[r];
        __syncthreads();
        pset ^= 1;
    };
    // out = src - lam dir (dir may be NULL: out = src), optionally truncated at 0; then a grid barrier
    auto update = [&](const float *src, const float *dir, float lam, int clip, float *out) {
        const size_t i0 = (size_t)blockIdx.x * nthr + tid, step = (size_t)nblk * nthr;
        const bool vec = p.nvox % 4 == 0 && ((uintptr_t)src % 16 == 0) && ((uintptr_t)out % 16 == 0) && (!dir || (uintptr_t)dir % 16 == 0);
        if (vec) {
            for (size_t o = i0; o < p.nvox / 4; o += step) {
                float4 v = ld_stream4(reinterpret_cast<const float4 *>(src) + o);
                if (dir) {
                    const float4 w = ld_stream4(reinterpret_cast<const float4 *>(dir) + o);
                    v.x = fmaf(-lam, w.x, v.x); v.y = fmaf(-lam, w.y, v.y); v.z = fmaf(-lam, w.z, v.z); v.w = fmaf(-lam, w.w, v.w);
                }
                if (clip) {
                    v.x = v.x < 0.0f ? 0.0f : v.x; v.y = v.y < 0.0f ? 0.0f : v.y;
                    v.z = v.z < 0.0f ? 0.0f : v.z; v.w = v.w < 0.0f ? 0.0f : v.w;
                }
                reinterpret_cast<float4 *>(out)[o] = v;
            }
        } else {
            for (size_t o = i0; o < p.nvox; o += step) {
                const float v = dir ? fmaf(-lam, dir[o], src[o]) : src[o];
                out[o] = (clip && v < 0.0f) ? 0.0f : v;
            }
        }
        grid.sync();
    };

    const float *cur = p.g;
    int which = 0, inner = 0, trials = 0;
    double E0 = 0.0, e_first = 0.0, e_last = 0.0;
    bool have_E0 = false, clipped = false;
    for (int it = 0; it < p.max_inner; ++it) {
        double tot[3];
        for (int t = next_tile(); t < ntiles; t = next_tile()) {
            double a0 = 0.0, a1 = 0.0, a2 = 0.0;
            const int tx = t % p.ntx, ty = (t / p.ntx) % p.nty, tz = t / (p.ntx * p.nty);
            if (VEC) {
                const TqTile T = tq_tile(p.D, p.zc, tx, ty, tz);
                if (cur == p.g) tq_grad_tile_async<true>(p.D, T, cur, p.g, (float)p.beta, p.delta2, p.d, tq_ring_base(), a0, a1, a2);
                else tq_grad_tile_async<false>(p.D, T, cur, p.g, (float)p.beta, p.delta2, p.d, tq_ring_base(), a0, a1, a2);
            } else {
                const TvTile T = tv_tile(p.D, p.zc, tx, ty, tz);
                if (cur == p.g) tv_grad_tile<true>(p.D, T, cur, p.g, (float)p.beta, p.delta2, p.d, a0, a1, a2);
                else tv_grad_tile<false>(p.D, T, cur, p.g, (float)p.beta, p.delta2, p.d, a0, a1, a2);
            }
            publish(t, a0, a1, a2, 3);
        }
        grid_sums(3, tot);
        if (!have_E0) { E0 = tot[0] / p.n + 0.5 * p.beta * tot[1] / p.n; e_first = e_last = E0; have_E0 = true; }
        const double Dm = tot[2] / p.n;
        double lam = 1.0 / p.beta, Enew = E0;
        bool accepted = false;
        float *cand = cur != p.f ? p.f : nullptr;           // the trial also leaves its (truncated) volume in f unless f is what it reads
        for (int bt = 0; bt <= p.max_bt; ++bt) {
            for (int t = next_tile(); t < ntiles; t = next_tile()) {
                double a0 = 0.0, a1 = 0.0;
                const int tx = t % p.ntx, ty = (t / p.ntx) % p.nty, tz = t / (p.ntx * p.nty);
                if (VEC) {
                    const TqTile T = tq_tile(p.D, p.zc, tx, ty, tz);
                    tq_energy_tile<true>(p.D, T, cur, p.d, p.g, (float)lam, p.delta2, cand, p.nonneg, a0, a1);
                } else {
                    const TvTile T = tv_tile(p.D, p.zc, tx, ty, tz);
                    tv_energy_tile<true>(p.D, T, cur, p.d, p.g, (float)lam, p.delta2, cand, p.nonneg, a0, a1);
                }
                publish(t, a0, a1, 0.0, 2);
            }
            double tr[3];
            grid_sums(2, tr);
            Enew = tr[0] / p.n + 0.5 * p.beta * tr[1] / p.n;
            ++trials;
            if (Enew <= E0 - p.armijo_c * lam * Dm) { accepted = true; break; }
            lam *= p.alpha;
        }
        if (!accepted) break;
        const double rel = fabs(Enew - E0) / E0;
        const bool last = rel < p.rel_tol || it + 1 == p.max_inner;
        float *nxt = last ? p.f : (which ? p.f2 : p.f);     // f, f2, f, ...: never cur unless last (in place is fine)
        which ^= 1;
        if (!(last && cur != p.f)) update(cur, p.d, (float)lam, last ? p.nonneg : 0, nxt);   // else the accepted trial wrote it
        cur = nxt;
        clipped = last;
        ++inner;
        E0 = Enew;
        e_last = Enew;
        if (last) break;
    }
    if (cur != p.f || (p.nonneg && !clipped)) update(cur, nullptr, 0.0f, p.nonneg, p.f);
    if (blockIdx.x == 0 && tid == 0) {
        p.report[0] = (double)inner; p.report[1] = (double)trials; p.report[2] = e_first; p.report[3] = e_last;
        p.report[4] += (double)inner; p.report[5] += (double)trials;
    }
}

// The 16-byte tiles need whole 16-byte groups per row and aligned rows; below 128 voxels per row they would idle lanes.
static bool tv_vec_ok(const cbct_geometry *g, const TvDims &D, const void *a, const void *b = nullptr, const void *c = nullptr,
                      const void *d = nullptr)
{
    if (g->tv_scalar_tiles) return false;
    if (D.nx % TQ_V != 0 || D.nx < TQ_W) return false;
    const void *p[4] = {a, b, c, d};
    for (int i = 0; i < 4; ++i)
        if (p[i] && (uintptr_t)p[i] % (4 * TQ_V) != 0) return false;
    return true;
}

// blocks of the cooperative kernel resident per SM (the register cap of its launch bounds decides)
// dynamic shared memory of the kernels that run the 16-byte gradient tiles (the cp.async rings); set once per kernel
static int tv_vec_smem() { return TQ_SMEM_PER_BLOCK; }
template <typename K> static bool tv_allow_smem(K kern)
{
    return tv_vec_smem() <= 48 * 1024 || cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, tv_vec_smem()) == cudaSuccess;
}

static int tv_coop_occupancy(bool vec)
{
    static int occs[2] = {0, 0};
    int &occ = occs[vec ? 1 : 0];
    if (occ == 0) {
        if (vec && !tv_allow_smem(tv_prox_coop_kernel<true>)) { cudaGetLastError(); return 0; }
        cudaError_t e = vec ? cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, tv_prox_coop_kernel<true>, 32 * TV_WPB, tv_vec_smem())
                            : cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, tv_prox_coop_kernel<false>, 32 * TV_WPB, 0);
        if (e != cudaSuccess) { cudaGetLastError(); occ = 0; return 0; }
    }
    return occ;
}

// The z-extent of a tile (the `zc` argument of the tile functions), the same for the cooperative kernel and for the passes as
// kernels of their own, so that both add the same per-tile partial sums.
//  * 32-voxel tiles: zc slices per tile; long marches amortise the halo slice and the block reduction, short ones keep every
//    SM supplied on small volumes (at least ~8 tiles per SM).
//  * 128-voxel tiles: the NUMBER of balanced z-chunks, fitted to the blocks resident at once: with chunks of about 16 slices
//    the tiles need m rounds of the persistent grid, and the chunk count is the largest that still fits m rounds -- at 256^3:
//    592 blocks, 32 tiles per chunk -> 18 chunks of 14-15 slices, one round (16 chunks of 16 would leave 80 blocks idle,
//    19 would need a second round for 16 tiles).
static int tv_zchunk(const cbct_geometry *g, const TvDims &D, bool vec)
{
    if (vec) {
        const long bxy = (long)((D.nx + TQ_W - 1) / TQ_W) * ((D.ny + TQ_R * TV_WPB - 1) / (TQ_R * TV_WPB));
        const long slots = (long)g->sm_count * (tv_coop_occupancy(true) > 0 ? tv_coop_occupancy(true) : 1);
        const long base = (D.nz + 15) / 16;
        const long m = (bxy * base + slots - 1) / slots;
        long ntz = m * slots / bxy;
        const long cap = D.nz >= 8 ? D.nz / 4 : 1;
        if (ntz > cap) ntz = cap;
        if (ntz < 1) ntz = 1;
        return (int)ntz;
    }
    const int bxy = ((D.nx + 31) / 32) * ((D.ny + TV_R * TV_WPB - 1) / (TV_R * TV_WPB));
    int zc = 32;
    while (zc > 4 && (long)bxy * ((D.nz + zc - 1) / zc) < 8L * g->sm_count) zc >>= 1;
    return zc;
}

static dim3 tv_grid(const TvDims &D, int zc, bool vec)
{
    if (vec) return dim3((D.nx + TQ_W - 1) / TQ_W, (D.ny + TQ_R * TV_WPB - 1) / (TQ_R * TV_WPB), zc);
    return dim3((D.nx + 31) / 32, (D.ny + TV_R * TV_WPB - 1) / (TV_R * TV_WPB), (D.nz + zc - 1) / zc);
}

static cbct_status launch_update(const cbct_geometry *g, size_t n, const float *f, const float *d, float lam, int clip,
                                 float *out, cudaStream_t st)
{
    const bool vec = n % 4 == 0 && ((uintptr_t)f % 16 == 0) && ((uintptr_t)out % 16 == 0) && (!d || (uintptr_t)d % 16 == 0);
    const int blocks = g->sm_count * 8;
    if (vec)
        tv_update_kernel<float4><<<blocks, 256, 0, st>>>(n / 4, reinterpret_cast<const float4 *>(f),
                                                         reinterpret_cast<const float4 *>(d), lam, clip,
                                                         reinterpret_cast<float4 *>(out));
    else
        tv_update_kernel<float><<<blocks, 256, 0, st>>>(n, f, d, lam, clip, out);
    CBCT_LAUNCH_CHECK(g);
    return CBCT_OK;
}

cbct_status launch_tv_energy(const cbct_geometry *g, const Level &L, const float *d_f, double delta,
                             double *d_out, cudaStream_t st)
{
    TvDims D = tv_dims(L);
    const bool vec = tv_vec_ok(g, D, d_f);
    const int zc = tv_zchunk(g, D, vec);
    dim3 gr = tv_grid(D, zc, vec), b(32, TV_WPB);
    if ((size_t)gr.x * gr.y * gr.z > (size_t)g->partials_stride)
        return cbct_fail(CBCT_ERR_INVALID_ARG, "volume too large for the reduction buffer");
    StageTimer t(g, st, ST_REDUCE);
    if (vec)
        tv_energy_kernel<false, true><<<gr, b, 0, st>>>(D, d_f, nullptr, nullptr, 0.0f, (float)(delta * delta), zc, 1,
                                                        g->d_partials, g->partials_stride, g->d_counter, d_out, nullptr, 0);
    else
        tv_energy_kernel<false, false><<<gr, b, 0, st>>>(D, d_f, nullptr, nullptr, 0.0f, (float)(delta * delta), zc, 1,
                                                         g->d_partials, g->partials_stride, g->d_counter, d_out, nullptr, 0);
    CBCT_LAUNCH_CHECK(g);
    return CBCT_OK;
}

// The cooperative kernel's launch: a grid of as many blocks as are resident at once.  The report (inner, trials, E_first,
// E_last) lands in d_scalars[16..19]; d_scalars[20..21] accumulate the counts over calls (cbct_fbs_reconstruct zeroes them).
static cbct_status launch_tv_prox_coop(const cbct_geometry *g, const Level &L, const float *d_g, float *d_f, double w,
                                       int nonneg, const cbct_tv_params &tp, cudaStream_t st)
{
    TvCoop p;
    p.D = tv_dims(L);
    const bool vec = tv_vec_ok(g, p.D, d_g, d_f, L.d_f2, L.d_d);
    const int occ = tv_coop_occupancy(vec);
    if (occ < 1) return cbct_fail(CBCT_ERR_CUDA, "the cooperative TV-prox kernel does not fit an SM");
    p.zc = tv_zchunk(g, p.D, vec);
    const dim3 tg = tv_grid(p.D, p.zc, vec);
    p.ntx = tg.x; p.nty = tg.y; p.ntz = tg.z;
    p.g = d_g; p.f = d_f; p.f2 = L.d_f2; p.d = L.d_d;
    p.beta = 1.0 / w; p.armijo_c = tp.armijo_c; p.alpha = tp.shrink_alpha; p.rel_tol = tp.rel_tol; p.n = (double)L.nvox;
    p.delta2 = (float)(tp.eps_delta * tp.eps_delta);
    p.max_inner = tp.max_inner; p.max_bt = tp.max_backtracks; p.nonneg = nonneg;
    p.nvox = L.nvox;
    p.partials = g->d_partials; p.stride = g->partials_stride;
    p.ticket = g->d_counter + 1;
    p.report = g->d_scalars + 16;
    long blocks = (long)g->sm_count * occ;
    const long ntiles = (long)tg.x * tg.y * tg.z;
    if (blocks > ntiles) blocks = ntiles;
    if (ntiles > g->partials_stride) return cbct_fail(CBCT_ERR_INVALID_ARG, "volume too large for the reduction buffer");
    void *args[] = {&p};
    StageTimer t(g, st, ST_TV_GRAD);
    const void *kern = vec ? (const void *)tv_prox_coop_kernel<true> : (const void *)tv_prox_coop_kernel<false>;
    CBCT_CUDA(cudaLaunchCooperativeKernel(kern, dim3((unsigned)blocks), dim3(32, TV_WPB), args, vec ? tv_vec_smem() : 0, st));
    CBCT_LAUNCH_CHECK(g);
    return CBCT_OK;
}

// Host-sequenced control loop (the Armijo test needs two global sums per trial).  The gradient pass
// and the first trial (its step 1/beta is known beforehand) are queued back to back and read with
// ONE stream synchronisation; the accepted update carries the non-negativity truncation when the
// stopping rule already says it is the last.  Scalars: d_scalars[0..2] gradient-pass sums,
// d_scalars[4..5] trial sums.
cbct_status run_tv_prox(const cbct_geometry *g, const Level &L, const float *d_g, float *d_f, double w,
                        int nonneg, const cbct_tv_params &tp, cbct_tv_report *rep, bool sync_report,
                        cudaStream_t st, TvAhead *ahead)
{
    if (ahead) ahead->valid = false;
    cbct_tv_report r = {0, 0, 0.0, 0.0};
    const size_t n = L.nvox;
    cbct_status s;
    if (w <= 0.0 || tp.max_inner == 0) {
        StageTimer t(g, st, ST_TV_UPDATE);
        if ((s = launch_update(g, n, d_g, nullptr, 0.0f, nonneg, d_f, st)) != CBCT_OK) return s;
        if (rep) *rep = r;
        return CBCT_OK;
    }
    if (!g->host_armijo) {
        // the whole call is one cooperative kernel; its report is read only when the caller wants it now
        if ((s = launch_tv_prox_coop(g, L, d_g, d_f, w, nonneg, tp, st)) != CBCT_OK) return s;
        if (rep && sync_report) {
            CBCT_CUDA(cudaMemcpyAsync(g->h_scalars + 16, g->d_scalars + 16, 4 * sizeof(double), cudaMemcpyDeviceToHost, st));
            CBCT_CUDA(cudaStreamSynchronize(st));
            r.inner_iters = (int)(g->h_scalars[16] + 0.5); r.trials = (int)(g->h_scalars[17] + 0.5);
            r.e_first = g->h_scalars[18]; r.e_last = g->h_scalars[19];
        }
        if (rep) *rep = r;
        return CBCT_OK;
    }
    TvDims D = tv_dims(L);
    const bool vec = tv_vec_ok(g, D, d_g, d_f, L.d_f2, L.d_d);
    const int zc = tv_zchunk(g, D, vec);
    dim3 gr = tv_grid(D, zc, vec), b(32, TV_WPB);
    const int S = g->partials_stride;
    if ((size_t)gr.x * gr.y * gr.z > (size_t)S) return cbct_fail(CBCT_ERR_INVALID_ARG, "volume too large for the reduction buffer");
    const double beta = 1.0 / w, N = (double)n;
    const float delta2 = (float)(tp.eps_delta * tp.eps_delta);
    double *ds = g->d_scalars, *hs = g->h_scalars;
    // ping-pong: cur holds f; the first f is g itself (read-only), later ones alternate
    const float *cur = d_g;
    float *bufs[2] = {d_f, L.d_f2};
    int which = 0;
    double E0 = 0.0;
    bool have_E0 = false, clipped = false;
    for (int it = 0; it < tp.max_inner; ++it) {
        {
            StageTimer t(g, st, ST_TV_GRAD);
            if (vec && !(tv_allow_smem(tv_grad_kernel<true, true>) && tv_allow_smem(tv_grad_kernel<false, true>)))
                return cbct_fail(CBCT_ERR_CUDA, "the gradient pass's shared-memory rings do not fit");
            if (cur == d_g && vec) tv_grad_kernel<true, true><<<gr, b, tv_vec_smem(), st>>>(D, cur, d_g, (float)beta, delta2, L.d_d, zc, g->d_partials, S, g->d_counter, ds);
            else if (cur == d_g) tv_grad_kernel<true, false><<<gr, b, 0, st>>>(D, cur, d_g, (float)beta, delta2, L.d_d, zc, g->d_partials, S, g->d_counter, ds);
            else if (vec) tv_grad_kernel<false, true><<<gr, b, tv_vec_smem(), st>>>(D, cur, d_g, (float)beta, delta2, L.d_d, zc, g->d_partials, S, g->d_counter, ds);
            else tv_grad_kernel<false, false><<<gr, b, 0, st>>>(D, cur, d_g, (float)beta, delta2, L.d_d, zc, g->d_partials, S, g->d_counter, ds);
            CBCT_LAUNCH_CHECK(g);
        }
        double lam = 1.0 / beta, Enew = E0, Dm = 0.0;
        bool accepted = false;
        int accepted_bt = -1;
        for (int bt = 0; bt <= tp.max_backtracks; ++bt) {
            {
                StageTimer t(g, st, ST_TV_TRIAL);
                // the trial also leaves its (truncated) volume in d_f unless d_f is what it reads
                if (vec)
                    tv_energy_kernel<true, true><<<gr, b, 0, st>>>(D, cur, L.d_d, d_g, (float)lam, delta2, zc, 2, g->d_partials, S,
                                                                   g->d_counter, ds + 4, cur != d_f ? d_f : nullptr, nonneg);
                else
                    tv_energy_kernel<true, false><<<gr, b, 0, st>>>(D, cur, L.d_d, d_g, (float)lam, delta2, zc, 2, g->d_partials, S,
                                                                    g->d_counter, ds + 4, cur != d_f ? d_f : nullptr, nonneg);
                CBCT_LAUNCH_CHECK(g);
            }
            CBCT_CUDA(cudaMemcpyAsync(hs, ds, 6 * sizeof(double), cudaMemcpyDeviceToHost, st));
            if (ahead && it == 0 && bt == 0) {
                // the candidate result is in d_f: let the caller queue what follows a successful prox behind this trial,
                // then wait for the trial's sums only -- the device keeps working while the host decides
                CBCT_CUDA(cudaEventRecord(g->ev[4], st));
                if ((s = ahead->fn(ahead->ctx)) != CBCT_OK) return s;
                CBCT_CUDA(cudaEventSynchronize(g->ev[4]));
            } else {
                CBCT_CUDA(cudaStreamSynchronize(st));
            }
            if (bt == 0) {
                if (!have_E0) { E0 = hs[0] / N + 0.5 * beta * hs[1] / N; r.e_first = r.e_last = E0; have_E0 = true; }
                Dm = hs[2] / N;
            }
            Enew = hs[4] / N + 0.5 * beta * hs[5] / N;
            ++r.trials;
            if (Enew <= E0 - tp.armijo_c * lam * Dm) { accepted = true; accepted_bt = bt; break; }
            lam *= tp.shrink_alpha;
        }
        if (!accepted) break;
        const double rel = fabs(Enew - E0) / E0;
        const bool last = rel < tp.rel_tol || it + 1 == tp.max_inner;
        float *nxt = last ? d_f : bufs[which];      // d_f, d_f2, d_f, ...: never cur unless last (in place is fine)
        which ^= 1;
        // the work queued behind the FIRST trial saw that trial's candidate: it is good only if that very trial was the
        // accepted one (a backtracked step has since overwritten d_f with another candidate) and the step is the last
        if (ahead && it == 0 && last && accepted_bt == 0) ahead->valid = true;
        if (!(last && cur != d_f)) {                 // else the accepted trial already wrote max(f - lam d, 0) to d_f
            StageTimer t(g, st, ST_TV_UPDATE);
            if ((s = launch_update(g, n, cur, L.d_d, (float)lam, last ? nonneg : 0, nxt, st)) != CBCT_OK) return s;
        }
        cur = nxt;
        clipped = last;
        ++r.inner_iters;
        E0 = Enew;
        r.e_last = Enew;
        if (last) break;
    }
    // result to d_f, with the non-negativity truncation, if the last update did not already do both
    if (cur != d_f || (nonneg && !clipped)) {
        StageTimer t(g, st, ST_TV_UPDATE);
        if ((s = launch_update(g, n, cur, nullptr, 0.0f, nonneg, d_f, st)) != CBCT_OK) return s;
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
