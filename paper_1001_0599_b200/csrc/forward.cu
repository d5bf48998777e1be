// forward.cu -- A1/A2: cone-beam forward projector, one thread per detector ray (or per group
// of four rays related by quarter turns of the gantry).
//
// (P f)[ray] = sum_voxels len(ray ∩ voxel) f[voxel]   (Eq. 1 on piecewise-
// constant voxels; "a ray-tracing algorithm, such as Siddon's", L187, L243).
//
// Instead of Siddon's data-dependent merge of three crossing lists, the ray is cut into unit
// slabs of its DRIVING axis (the in-plane axis along which it crosses more planes).  Inside one
// slab it crosses at most one plane of the other in-plane axis and at most one z-plane (checked
// at create), so it touches at most three voxels whose lengths follow in closed form from the
// two crossing parameters sy, sz in [0,1]:  min(sy,sz), |sy-sz|, 1-max(sy,sz).  These are the
// exact radiological path -- Siddon's numbers up to rounding -- but every thread of a warp runs
// the same branch-free loop.
//
// Memory: the volume is staged once per projection into a zero-padded copy with z FASTEST,
// [i][j][k], and the 32 lanes of a warp are 32 consecutive detector ROWS of one detector column.
// All lanes then share the in-plane path (same slab, same minor cell, same in-plane crossing) and
// differ only in z, where their cells are consecutive: every load of the warp falls in one or two
// 128-byte lines whatever the view angle, one copy serves both driving axes and all quarter turns
// (it stays L2-resident), and no load needs a bounds test (cbct_internal.cuh, PAD_M / PAD_Z).  The
// cell of the ray is tracked incrementally (the next plane on each axis and a linear offset), so
// the loop holds no floor, no integer multiply and no divergent branch.
//
// Mirror symmetry (nmir == 2): with the volume centred in z and the detector centred in v, the ray
// (iu, nv-1-iv) is the mirror image z -> -z of the ray (iu, iv); the same thread walks it through
// the cells nz-1-k with the same weights.
//
// Rotation symmetry (nsym == 4): on a square, centred in-plane grid with views at angles
// t, t+90, t+180, t+270 degrees, the ray (t + 90 r, iu, iv) is the ray (t, iu, iv) turned by
// r quarter turns, and a quarter turn maps voxel (i,j) to (n-1-j, i).  One thread then walks
// the base ray once and applies its weights to the four turned copies of the cell: the crossing
// arithmetic is shared, only the loads and FMAs are per view.
#include "cbct_internal.cuh"
#include "ray.cuh"
#include "reduce.cuh"

// vol [k][j][i] -> stage[i+PM][j+PM][k+PZ]: per j, a 32x32 (k,i) tile through shared memory.
// The margins of the staged copy were zeroed at create and are never written.
__global__ void stage_volume_kernel(const float *__restrict__ in, float *__restrict__ stage, int nx, int ny, int nz,
                                    int istride, int jstride)
{
    __shared__ float tile[32][33];
    const int j = blockIdx.z;
    const int i = blockIdx.x * 32 + threadIdx.x, k0 = blockIdx.y * 32;
    for (int r = threadIdx.y; r < 32; r += blockDim.y) {
        const int k = k0 + r;
        if (i < nx && k < nz) tile[r][threadIdx.x] = __ldg(in + ((size_t)k * ny + j) * nx + i);
    }
    __syncthreads();
    const int k = k0 + threadIdx.x, i0 = blockIdx.x * 32;
    for (int r = threadIdx.y; r < 32; r += blockDim.y) {
        const int ii = i0 + r;
        if (ii < nx && k < nz)
            stage[(size_t)(ii + PAD_M) * istride + (size_t)(j + PAD_M) * jstride + k + PAD_Z] = tile[threadIdx.x][r];
    }
}

// Mirror-packed staging (nmir == 2): stage2[i+PM][j+PM][kk] = ( f(i,j,k), f(i,j,nz-1-k) ), k = kk - PZ, for
// kk in [0, nz/2 + 2 PZ); a component whose k falls outside the grid is 0.  A ray of the lower detector half and
// its mirror image then read their two cells with ONE 8-byte load at the same offset.  (The entries with
// k >= nz/2 repeat pairs with the roles swapped: the one-cell slack of the incremental cell tracking may touch
// k = nz/2 with weight 0.)  Every element of the copy, margins included, is written here.
__global__ void stage_volume_packed_kernel(const float *__restrict__ in, float2 *__restrict__ stage, int nx, int ny,
                                           int nz, int istride, int jstride)
{
    __shared__ float lo[32][33], hi[32][33];
    const int j = blockIdx.z;
    const int i = blockIdx.x * 32 + threadIdx.x, kk0 = blockIdx.y * 32;
    for (int r = threadIdx.y; r < 32; r += blockDim.y) {
        const int k = kk0 + r - PAD_Z, km = nz - 1 - k;
        float a = 0.0f, b = 0.0f;
        if (i < nx) {
            if (k >= 0 && k < nz) a = __ldg(in + ((size_t)k * ny + j) * nx + i);
            if (km >= 0 && km < nz) b = __ldg(in + ((size_t)km * ny + j) * nx + i);
        }
        lo[r][threadIdx.x] = a; hi[r][threadIdx.x] = b;
    }
    __syncthreads();
    const int kk = kk0 + threadIdx.x, i0 = blockIdx.x * 32;
    for (int r = threadIdx.y; r < 32; r += blockDim.y) {
        const int ii = i0 + r;
        if (ii < nx && kk < jstride)
            stage[(size_t)(ii + PAD_M) * istride + (size_t)(j + PAD_M) * jstride + kk] =
                make_float2(lo[threadIdx.x][r], hi[threadIdx.x][r]);
    }
}

// The same copy with 16-byte accesses on both sides (nx % 4 == 0, nzP even): a block takes one j, 64 voxels in i and 32
// cells in kk; a half warp reads a 256-byte row of the volume with one float4 per lane, and writes 32 consecutive cells of a
// staged column (256 bytes) with one float4 = two cells per lane.  Ten times fewer instructions per cell than the kernel
// above, which was issue bound (0.054 ms at 256^3, 36 M warp instructions).
constexpr int STG_I = 64, STG_K = 32;
__global__ void __launch_bounds__(256)
stage_volume_packed_vec_kernel(const float *__restrict__ in, float4 *__restrict__ stage2, int nx, int ny, int nz,
                               int istride, int jstride)
{
    __shared__ float lo[STG_K][STG_I + 1], hi[STG_K][STG_I + 1];
    const int j = blockIdx.z, i0 = blockIdx.x * STG_I, kk0 = blockIdx.y * STG_K;
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    {
        const int c = lane & 15, i = i0 + 4 * c;
#pragma unroll
        for (int pass = 0; pass < 2; ++pass) {
            const int r = pass * 16 + warp * 2 + (lane >> 4);
            const int k = kk0 + r - PAD_Z, km = nz - 1 - k;
            float4 a = make_float4(0.f, 0.f, 0.f, 0.f), b = a;
            if (i < nx && k >= 0 && k < nz) {                    // km is in range exactly when k is
                a = __ldg(reinterpret_cast<const float4 *>(in + ((size_t)k * ny + j) * nx + i));
                b = __ldg(reinterpret_cast<const float4 *>(in + ((size_t)km * ny + j) * nx + i));
            }
            lo[r][4 * c + 0] = a.x; lo[r][4 * c + 1] = a.y; lo[r][4 * c + 2] = a.z; lo[r][4 * c + 3] = a.w;
            hi[r][4 * c + 0] = b.x; hi[r][4 * c + 1] = b.y; hi[r][4 * c + 2] = b.z; hi[r][4 * c + 3] = b.w;
        }
    }
    __syncthreads();
    const int kl = 2 * (lane & 15), kk = kk0 + kl;               // this lane's two cells
#pragma unroll
    for (int pass = 0; pass < 4; ++pass) {
        const int il = pass * 16 + warp * 2 + (lane >> 4), ii = i0 + il;
        if (ii < nx && kk < jstride) {                          // jstride = nzP is even: kk + 1 < nzP too
            const size_t cell = (size_t)(ii + PAD_M) * istride + (size_t)(j + PAD_M) * jstride + kk;
            stage2[cell >> 1] = make_float4(lo[kl][il], hi[kl][il], lo[kl + 1][il], hi[kl + 1][il]);
        }
    }
}

constexpr int FWD_BV = 32, FWD_BU = 8;      // block: 32 detector rows (lanes) x 8 detector columns
#ifndef FWD_MINB
#define FWD_MINB 2
#endif

// One staged cell: a voxel value (M == 1) or the mirror pair (f(k), f(nz-1-k)) (M == 2).
template <int M> struct StageCell { typedef float type; };
template <> struct StageCell<2> { typedef float2 type; };
__device__ __forceinline__ float cell_lo(float c) { return c; }
__device__ __forceinline__ float cell_lo(float2 c) { return c.x; }
__device__ __forceinline__ float cell_hi(float c) { return c; }
__device__ __forceinline__ float cell_hi(float2 c) { return c.y; }

// What a walk leaves behind: the RF * M sums of a thread's rays (acc[mm * R * F + fl * R + q]: mirror image mm, reflection fl,
// quarter turn q of the walk) scaled to line integrals and written as MODE says; returns through sq the squared residuals.
template <int R, int M, int MODE, int F>
__device__ __forceinline__ void forward_epilogue(const LevelParams &P, const RayU &r, float v, const float (&acc)[R * F * M], int a, int ar,
                                                 int iu, int iv, const float *__restrict__ y, float *__restrict__ out, double &sq)
{
    constexpr int RF = R * F;
    const float Lr = ray_len_L(r, v);
    const float scale = Lr * r.inv_dd;
    const size_t plane = (size_t)P.nv * P.nu;
#pragma unroll
    for (int mm = 0; mm < M; ++mm) {
        const int ivm = mm ? P.nv - 1 - iv : iv;
#pragma unroll
        for (int fl = 0; fl < F; ++fl) {                // the walk's own rays, then their reflections
            const int av = fl ? ar : a, iuv = fl ? P.nu - 1 - iu : iu;
            const size_t pix = (size_t)ivm * P.nu + iuv;
            float res[R];
#pragma unroll
            for (int q = 0; q < R; ++q) {
                // the quarter turn of view `av` this image belongs to
                const int qv = fl ? ((a == 0 ? 4 - q : 3 - q) & 3) : q;
                const float pr = acc[mm * RF + fl * R + q] * scale;
                const size_t o1 = (size_t)(av + qv * P.nbase) * plane + pix;
                float val = 0.0f;
                if (MODE == 0) {
                    out[o1] = pr;
                } else if (MODE == 4) {                // plain residual for the Eq. 6 back-projector
                    const float T = pr - __ldg(y + o1);
                    out[o1] = T;
                    sq += (double)T * (double)T;
                } else if (MODE == 2) {
                    val = pr * scale;                  // L inv_dd * (P f): input of the transpose without a residual
                } else {
                    const float T = pr - __ldg(y + o1);
                    val = T * scale;                   // what the transpose consumes (see back.cu)
                    sq += (double)T * (double)T;
                }
                // position of this quarter turn in the interleaved entry (a compile-time permutation per a == 0 or not)
                if (!fl) res[q] = val;
                else if (a == 0) res[(4 - q) & 3 & (R - 1)] = val;
                else res[(3 - q) & 3 & (R - 1)] = val;
            }
            if (MODE != 0 && MODE != 4) {              // d_T layout: [base view][iu][iv] (x4 interleaved)
                const size_t ot = ((size_t)av * P.nu + iuv) * P.nv + t_row_slot(P, ivm);
                if (R == 4) reinterpret_cast<float4 *>(out)[ot] = make_float4(res[0], res[1 % R], res[2 % R], res[3 % R]);
                else out[ot] = res[0];
            }
        }
    }
}

// R = quarter-turn views per thread (1 or 4), M = 2 when the thread also walks the mirror image
// z -> -z of its ray (detector row nv-1-iv, cells nz-1-k): same weights again, and -- the staged
// copy being mirror-packed -- the same loads.  MODE as in launch_forward.
// F = 2 (with R == 4 only): the thread also walks the REFLECTIONS y -> -y of its four rays.  On a view set that is symmetric
// under theta -> -theta (theta_0 = 0, detector centred in u, nu even) the reflected ray of (base view a, quarter turn q, column
// iu) is (base view (n_base - a) % n_base, quarter turn (3 - q) % 4 -- (4 - q) % 4 for a = 0 --, column nu-1-iu) and crosses
// the cells (i, ny-1-j) with the same weights: one walk then serves 16 rays.  The grid's y dimension counts view PAIRS
// p = 0 .. n_base/2; the self-paired views (p = 0, and p = n_base/2 when n_base is even) walk the columns iu < nu/2 only.
template <int R, int M, int MODE, int F>
__global__ void __launch_bounds__(FWD_BV *FWD_BU, FWD_MINB)
forward_kernel(const LevelParams P, const void *__restrict__ stage_v, const RayU *__restrict__ rayu,
               const float *__restrict__ y, float *__restrict__ out, double *__restrict__ partials, int stride,
               unsigned int *__restrict__ counter, double *__restrict__ sum_out, int a_off)
{
    typedef typename StageCell<M>::type cell;
    const cell *__restrict__ stage = reinterpret_cast<const cell *>(stage_v);
    __shared__ double slot[32];
    // detector-row tiles are the slowest grid dimension: the blocks in flight together then walk one z-slab of the
    // staged copy for every view, which stays in L2 (with the view slowest, every view re-reads the whole copy)
    const int iv = blockIdx.z * FWD_BV + threadIdx.x;
    const int iu = blockIdx.x * FWD_BU + threadIdx.y;
    const int a = blockIdx.y + a_off;          // base view, or view pair (a_off: first unit of a sharded launch)
    const int nvh = M == 2 ? P.nv / 2 : P.nv;  // rows this grid walks; the others are their mirrors
    constexpr int RF = R * F;                  // images of the walk in-plane
    const int ar = F == 2 ? (P.nbase - a) % P.nbase : a;                 // base view of the reflected rays
    const int nuw = (F == 2 && ar == a) ? P.nu / 2 : P.nu;               // columns this unit walks
    double sq = 0.0;
    if (iu < nuw && iv < nvh) {
        const RayU r = load_rayu(rayu, a * P.nu + iu);
        const float v = fmaf((float)iv, P.dv, P.v0);
        const RayZ rz = ray_z(r, v, P.sz);
        // driving axis: nd slabs; minor axis: nm voxels
        const int nd = r.drive ? P.ny : P.nx, nm = r.drive ? P.nx : P.ny;
        const int cd = r.drive ? P.cy : P.cx, cm = r.drive ? P.cx : P.cy;
        // slabs in which the ray comes within half a voxel of the volume
        float dlo = (float)(-cd), dhi = (float)(nd - cd);
        {
            const float t1 = ((float)(-cm) - 0.5f - r.a0) * r.inv_m, t2 = ((float)(nm - cm) + 0.5f - r.a0) * r.inv_m;
            dlo = fmaxf(dlo, fminf(t1, t2)); dhi = fminf(dhi, fmaxf(t1, t2));
            const float t3 = ((float)(-P.cz) - 0.5f - rz.za) * rz.inv_mz, t4 = ((float)(P.nz - P.cz) + 0.5f - rz.za) * rz.inv_mz;
            dlo = fmaxf(dlo, fminf(t3, t4)); dhi = fminf(dhi, fmaxf(t3, t4));
        }
        float acc[RF * M];
#pragma unroll
        for (int q = 0; q < RF * M; ++q) acc[q] = 0.0f;
        if (dhi > dlo) {
            const int s_lo = max(0, (int)floorf(dlo) + cd), s_hi = min(nd, (int)ceilf(dhi) + cd);
            float d = (float)(s_lo - cd);
            float y0 = fmaf(d, r.m, r.a0), z0 = fmaf(d, rz.mz, rz.za);
            const float fy = floorf(y0), fz = floorf(z0);
            const bool posy = r.m >= 0.0f, posz = rz.mz >= 0.0f;
            float nexty = posy ? fy + 1.0f : fy, nextz = posz ? fz + 1.0f : fz;
            const float sgny = posy ? 1.0f : -1.0f, sgnz = posz ? 1.0f : -1.0f;
            const int dj = posy ? 1 : -1, dk = posz ? 1 : -1;
            const int jm = (int)fy + cm, kk = (int)fz + P.cz + PAD_Z;
            // the current cell in (i,j), its slab step and its minor-axis step; a quarter turn maps
            // a position (i,j) -> (n-1-j, i) and a step (di,dj) -> (-dj, di)
            int ci = r.drive ? jm : s_lo, cj = r.drive ? s_lo : jm;
            int si = r.drive ? 0 : 1, sj = r.drive ? 1 : 0;
            int mi = r.drive ? dj : 0, mj = r.drive ? 0 : dj;
            int off[RF], drow[RF], dcol[RF];    // element offsets into the staged copy (< 2^31, checked at create)
#pragma unroll
            for (int q = 0; q < R; ++q) {
                off[q] = (ci + PAD_M) * P.istride + (cj + PAD_M) * P.jstride + kk;
                drow[q] = si * P.istride + sj * P.jstride;
                dcol[q] = mi * P.istride + mj * P.jstride;
                if (F == 2) {                   // the reflection y -> -y of this turned copy: cell (i, ny-1-j), steps (di, -dj)
                    off[R + q] = (ci + PAD_M) * P.istride + (P.ny - 1 - cj + PAD_M) * P.jstride + kk;
                    drow[R + q] = si * P.istride - sj * P.jstride;
                    dcol[R + q] = mi * P.istride - mj * P.jstride;
                }
                int t = ci; ci = P.nx - 1 - cj; cj = t;
                t = si; si = -sj; sj = t;
                t = mi; mi = -mj; mj = t;
            }
#ifdef FWD_UNROLL
#pragma unroll FWD_UNROLL
#endif
            for (int s = s_lo; s < s_hi; ++s) {
                // crossing parameters of the next minor-axis plane and the next z-plane, clipped to the slab
                const float sy = __saturatef((nexty - y0) * r.inv_m);
                const float sz = __saturatef((nextz - z0) * rz.inv_mz);
                const bool cy = sy < 1.0f, cz = sz < 1.0f;
                const float lo = fminf(sy, sz);                          // first cell: [0, lo]
                const float hi = (cy && cz) ? fmaxf(sy, sz) : lo;        // middle cell: [lo, hi]; last: [hi, 1]
                const float wl = 1.0f - hi;
                const int zc = cz ? dk : 0;
                // issue every load of the step before the first use: the loop is bound by load latency otherwise
                int offc[RF];
                cell va[RF], vc[RF];
#pragma unroll
                for (int q = 0; q < RF; ++q) offc[q] = off[q] + (cy ? dcol[q] : 0) + zc;
#pragma unroll
                for (int q = 0; q < RF; ++q) {
                    CBCT_DEV_ASSERT(off[q] >= 0 && off[q] < P.stage_cells && offc[q] >= 0 && offc[q] < P.stage_cells);
                    va[q] = __ldg(stage + off[q]); vc[q] = __ldg(stage + offc[q]);
                }
#pragma unroll
                for (int q = 0; q < RF; ++q) {
                    acc[q] = fmaf(wl, cell_lo(vc[q]), fmaf(lo, cell_lo(va[q]), acc[q]));
                    if (M == 2) acc[RF + q] = fmaf(wl, cell_hi(vc[q]), fmaf(lo, cell_hi(va[q]), acc[RF + q]));
                }
                if (hi > lo) {      // both planes crossed inside this slab, at different parameters (rare): a third cell
                    const float wm = hi - lo;
                    const bool yfirst = sy < sz;
#pragma unroll
                    for (int q = 0; q < RF; ++q) {
                        CBCT_DEV_ASSERT(off[q] + (yfirst ? dcol[q] : dk) >= 0 && off[q] + (yfirst ? dcol[q] : dk) < P.stage_cells);
                        const cell vm = __ldg(stage + off[q] + (yfirst ? dcol[q] : dk));
                        acc[q] = fmaf(wm, cell_lo(vm), acc[q]);
                        if (M == 2) acc[RF + q] = fmaf(wm, cell_hi(vm), acc[RF + q]);
                    }
                }
#pragma unroll
                for (int q = 0; q < RF; ++q) off[q] = offc[q] + drow[q];
                if (cy) nexty += sgny;
                if (cz) nextz += sgnz;
                d += 1.0f;
                y0 = fmaf(d, r.m, r.a0);
                z0 = fmaf(d, rz.mz, rz.za);
            }
        }
        forward_epilogue<R, M, MODE, F>(P, r, v, acc, a, ar, iu, iv, y, out, sq);
    }
    if (MODE == 1 || MODE == 4) {        // E2 numerator: sum of squared residuals, second stage fused (reduce.cuh)
        double s[1];
        s[0] = block_sum(sq, slot);
        if (counter) publish_and_finalize<1>(s, 1, partials, stride, counter, sum_out, slot);
        else publish_only<1>(s, 1, partials, stride, ((unsigned)blockIdx.z * (F == 2 ? P.npairs : P.nbase) + a) * gridDim.x + blockIdx.x);   // sharded launch
    }
}

// ---------------------------------------------------------------------------------------------------------------------------
// The FOLDED staged copy and its walk (quarter-turn + mirror symmetric levels: nsym == 4, nmir == 2).
//
// The 8 (16 with view pairs) rays of a thread read, in every cell (i, j, k) they cross, the cell's images under the quarter
// turns (and the reflection y -> -y) and under the mirror z -> -z.  forward_kernel fetches each image with its own 8-byte load at
// its own offset: per slab step of 16 rays, 16 loads + 16 address computations + 16 offset updates of 113 instructions.  Here
// the staged copy is folded onto the first quadrant instead: the entry of the canonical cell (i0, j0), i0, j0 < n/2, holds
//     E(i0, j0, kk) = ( f(R^q (i0, j0), k), q = 0..3 | f(R^q (i0, j0), nz-1-k), q = 0..3 ),   R (i, j) = (n-1-j, i),  k = kk - PZ
// -- two float4, each in a plane of its own (the lanes of a warp are consecutive detector rows: their entries are neighbours in kk,
// and a 16-byte load per lane at a 16-byte stride costs half the L1 wavefronts of one at a 32-byte stride), the same
// 8 n^2 nzP / 4 floats in all.  A cell (i, j) in quadrant m (m = 0: i, j < n/2; 1: i >= n/2 >
// j; 2: both >=; 3: j >= n/2 > i) is R^m of its canonical cell, so the q-th turned copy of the ray reads component (q + m) mod 4
// of ONE entry (two 16-byte loads); its reflection's q-th copy reads component (3 - q - m) mod 4 of the entry of the TRANSPOSED
// canonical cell (j0, i0) (S R^m (i0, j0) = R^(3-m) (j0, i0) with S the reflection).  A slab step of 16 rays is then 8 loads of
// 16 bytes at 4 offsets.  The sums are kept in the frame of the current quadrant (accumulator c belongs to component c) and
// rotated when the walk changes quadrant -- at the centre plane of the driving axis, between two slabs, and in the one slab
// where the ray crosses the centre plane of the minor axis, which takes a generic path (fold_cell); a walk changes quadrant
// at most three times.  Same weights as forward_kernel; the 8-ray walk adds them in the same order (the same bits), the
// view-pair walk adds the z-neighbour cells of slabs without an in-plane crossing in batches (FOLD_DEFER: equal to 4e-8).
// Margins: canonical coordinates run from -PAD_M (a cell outside the grid folds to a negative canonical coordinate); those
// entries, and the components of k outside the grid, are written as zeros by the staging kernel.

constexpr int FOLD_T = 16, FOLD_K = 8;       // staging tile: 16 x 16 canonical cells x 8 cells in kk of one half (k, or its mirror)
// vol [k][j][i] -> fold[half][(i0+PM)][(j0+PM)][kk] (float4): every image's 16 x 16 patch is read with x fastest (64-byte runs) and
// the tile leaves as 128-byte runs (8 entries of one canonical column).  blockIdx.z = 2 * (tile in kk) + half.
__global__ void __launch_bounds__(256)
stage_volume_fold_kernel(const float *__restrict__ in, float4 *__restrict__ fold, int n, int nz, int nhP, int nzP)
{
    __shared__ float tile[4][FOLD_K][FOLD_T][FOLD_T + 1];            // [q][kk][i0][j0]
    const int a0 = blockIdx.x * FOLD_T, b0 = blockIdx.y * FOLD_T, kk0 = (blockIdx.z >> 1) * FOLD_K, half = blockIdx.z & 1;
    const int tx = threadIdx.x & 15, ty = threadIdx.x >> 4, n1 = n - 1;
#pragma unroll
    for (int q = 0; q < 4; ++q) {
        // thread (tx, ty) of image q's patch: x runs with tx.  q = 0: (x, y) = (i0, j0); 1: (n1 - j0, i0); 2: (n1 - i0, n1 - j0);
        // 3: (j0, n1 - i0)
        int il, jl;
        if (q == 0) { il = tx; jl = ty; }
        else if (q == 1) { jl = FOLD_T - 1 - tx; il = ty; }
        else if (q == 2) { il = FOLD_T - 1 - tx; jl = FOLD_T - 1 - ty; }
        else { jl = tx; il = FOLD_T - 1 - ty; }
        const int i0 = a0 + il - PAD_M, j0 = b0 + jl - PAD_M;
        const int x = q == 0 ? i0 : q == 1 ? n1 - j0 : q == 2 ? n1 - i0 : j0;
        const int y = q == 0 ? j0 : q == 1 ? i0 : q == 2 ? n1 - j0 : n1 - i0;
        const bool inpl = i0 >= 0 && j0 >= 0 && i0 < n / 2 && j0 < n / 2;
#pragma unroll
        for (int c = 0; c < FOLD_K; ++c) {
            const int k = kk0 + c - PAD_Z, ks = half ? nz - 1 - k : k;       // the mirror is in range exactly when k is
            tile[q][c][il][jl] = (inpl && k >= 0 && k < nz) ? __ldg(in + ((size_t)ks * n + y) * n + x) : 0.0f;
        }
    }
    __syncthreads();
    const int c = threadIdx.x & 7;                                   // 8 float4 = 8 entries = 128 bytes per canonical column
#pragma unroll
    for (int it = 0; it < 8; ++it) {
        const int cell = (threadIdx.x >> 3) + 32 * it, il = cell >> 4, jl = cell & 15;
        const int a = a0 + il, b = b0 + jl, kk = kk0 + c;
        if (a < nhP && b < nhP && kk < nzP)
            fold[(size_t)half * nhP * nhP * nzP + ((size_t)a * nhP + b) * nzP + kk] =
                make_float4(tile[0][c][il][jl], tile[1][c][il][jl], tile[2][c][il][jl], tile[3][c][il][jl]);
    }
}

// frame rotations of four sums: up: new[(c + 1) & 3] = old[c]; down: new[(c - 1) & 3] = old[c]
__device__ __forceinline__ void fold_rot_up(float (&a)[4]) { const float t = a[3]; a[3] = a[2]; a[2] = a[1]; a[1] = a[0]; a[0] = t; }
__device__ __forceinline__ void fold_rot_dn(float (&a)[4]) { const float t = a[0]; a[0] = a[1]; a[1] = a[2]; a[2] = a[3]; a[3] = t; }
// component c of the result = component (c + d) & 3 of v
__device__ __forceinline__ float4 fold_rot4(float4 v, int d)
{
    if (d & 1) v = make_float4(v.y, v.z, v.w, v.x);
    if (d & 2) v = make_float4(v.z, v.w, v.x, v.y);
    return v;
}
__device__ __forceinline__ void fold_fma(float (&a)[4], float w, const float4 v)
{
    a[0] = fmaf(w, v.x, a[0]); a[1] = fmaf(w, v.y, a[1]); a[2] = fmaf(w, v.z, a[2]); a[3] = fmaf(w, v.w, a[3]);
}

// quadrant m of the cell (ci, cj) and its canonical cell (i0, j0): (ci, cj) = R^m (i0, j0)
__device__ __forceinline__ int fold_canon(int ci, int cj, int nh, int n1, int &i0, int &j0)
{
    const bool qi = ci >= nh, qj = cj >= nh;
    const int m = qi ? (qj ? 2 : 1) : (qj ? 3 : 0);
    i0 = m == 0 ? ci : m == 1 ? cj : m == 2 ? n1 - ci : n1 - cj;
    j0 = m == 0 ? cj : m == 1 ? n1 - ci : m == 2 ? n1 - cj : ci;
    return m;
}
// a step (di, dj) of the cell seen from the canonical cell of quadrant m
__device__ __forceinline__ void fold_step(int m, int di, int dj, int &d0i, int &d0j)
{
    d0i = m == 0 ? di : m == 1 ? dj : m == 2 ? -di : -dj;
    d0j = m == 0 ? dj : m == 1 ? -di : m == 2 ? -dj : di;
}

// One cell of the slab that crosses the centre plane of the minor axis: any quadrant, added into the sums kept in frame m.
template <int F>
__device__ __forceinline__ void fold_cell(const LevelParams &P, const float4 *__restrict__ fold, int ci, int cj, int kk, float w, int m,
                                          float (&accB)[2][4], float (&accT)[2][4])
{
    int i0, j0;
    const int mc = fold_canon(ci, cj, P.nx / 2, P.nx - 1, i0, j0);
    const int dlt = (mc - m) & 3;
    const int oB = (i0 + PAD_M) * P.fis + (j0 + PAD_M) * P.fjs + kk;
    CBCT_DEV_ASSERT(oB >= 0 && oB < P.stage_cells);
    const float4 *__restrict__ fold_hi = fold + P.stage_cells;
    const float4 b0 = __ldg(fold + oB), b1 = __ldg(fold_hi + oB);
    fold_fma(accB[0], w, fold_rot4(b0, dlt));
    fold_fma(accB[1], w, fold_rot4(b1, dlt));
    if (F == 2) {
        const int oT = (j0 + PAD_M) * P.fis + (i0 + PAD_M) * P.fjs + kk;
        CBCT_DEV_ASSERT(oT >= 0 && oT < P.stage_cells);
        const float4 t0 = __ldg(fold + oT), t1 = __ldg(fold_hi + oT);
        fold_fma(accT[0], w, fold_rot4(t0, (4 - dlt) & 3));
        fold_fma(accT[1], w, fold_rot4(t1, (4 - dlt) & 3));
    }
}

#ifndef FOLD_BU
#define FOLD_BU 8           // detector columns per block (x 32 rows)
#endif
#ifndef FOLD_MINB2
#define FOLD_MINB2 3        // resident blocks per SM the view-pair walk is compiled for (80 registers), and the 8-ray walk
#endif
#ifndef FOLD_MINB1
#define FOLD_MINB1 2
#endif
#ifndef FOLD_DEFER
#define FOLD_DEFER 1        // 1: the view-pair walk fetches the z-neighbour cell of a slab without an in-plane crossing in batches
#endif                      // (see the kernel; measured slower on the 8-ray walk: 0.682 against 0.637 ms at config 3)
// forward_kernel<4, 2, MODE, F> on the folded copy: same grid, same rays per thread, same epilogue.
template <int MODE, int F>
__global__ void __launch_bounds__(FWD_BV *FOLD_BU, F == 2 ? FOLD_MINB2 : FOLD_MINB1)
forward_fold_kernel(const LevelParams P, const float4 *__restrict__ fold, const RayU *__restrict__ rayu,
                    const float *__restrict__ y, float *__restrict__ out, double *__restrict__ partials, int stride,
                    unsigned int *__restrict__ counter, double *__restrict__ sum_out, int a_off)
{
    __shared__ double slot[32];
    const float4 *__restrict__ fold_hi = fold + P.stage_cells;     // the z-mirror components: a plane of their own
    const int iv = blockIdx.z * FWD_BV + threadIdx.x;
    const int iu = blockIdx.x * FOLD_BU + threadIdx.y;
    const int a = blockIdx.y + a_off;
    const int nvh = P.nv / 2;
    const int ar = F == 2 ? (P.nbase - a) % P.nbase : a;
    const int nuw = (F == 2 && ar == a) ? P.nu / 2 : P.nu;
    double sq = 0.0;
    if (iu < nuw && iv < nvh) {
        const RayU r = load_rayu(rayu, a * P.nu + iu);
        const float v = fmaf((float)iv, P.dv, P.v0);
        const RayZ rz = ray_z(r, v, P.sz);
        const int n = P.nx, nh = n / 2, n1 = n - 1;           // square, even, centred grid: cx = cy = nh
        float dlo = (float)(-nh), dhi = (float)(n - nh);
        {
            const float t1 = ((float)(-nh) - 0.5f - r.a0) * r.inv_m, t2 = ((float)(n - nh) + 0.5f - r.a0) * r.inv_m;
            dlo = fmaxf(dlo, fminf(t1, t2)); dhi = fminf(dhi, fmaxf(t1, t2));
            const float t3 = ((float)(-P.cz) - 0.5f - rz.za) * rz.inv_mz, t4 = ((float)(P.nz - P.cz) + 0.5f - rz.za) * rz.inv_mz;
            dlo = fmaxf(dlo, fminf(t3, t4)); dhi = fminf(dhi, fmaxf(t3, t4));
        }
        float accB[2][4], accT[2][4];                         // [mirror][component of the entry]: the frame of quadrant m
#pragma unroll
        for (int c = 0; c < 4; ++c) { accB[0][c] = accB[1][c] = 0.0f; accT[0][c] = accT[1][c] = 0.0f; }
        int m = 0;
        if (dhi > dlo) {
            const int s_lo = max(0, (int)floorf(dlo) + nh), s_hi = min(n, (int)ceilf(dhi) + nh);
            float d = (float)(s_lo - nh);
            float y0 = fmaf(d, r.m, r.a0), z0 = fmaf(d, rz.mz, rz.za);
            const float fy = floorf(y0), fz = floorf(z0);
            const bool posy = r.m >= 0.0f, posz = rz.mz >= 0.0f;
            float nexty = posy ? fy + 1.0f : fy, nextz = posz ? fz + 1.0f : fz;
            const float sgny = posy ? 1.0f : -1.0f, sgnz = posz ? 1.0f : -1.0f;
            const int dj = posy ? 1 : -1, dk = posz ? 1 : -1;
            const int si = r.drive ? 0 : 1, sj = r.drive ? 1 : 0;          // slab step and minor-axis step of the cell
            const int mi = r.drive ? dj : 0, mj = r.drive ? 0 : dj;
            int s = s_lo;
            while (s < s_hi) {
                // ---- a run of slabs inside one quadrant: the cell from the tracked planes, the sums turned into its frame ----
                const int jm = (int)nexty - (posy ? 1 : 0) + nh, kk = (int)nextz - (posz ? 1 : 0) + P.cz + PAD_Z;
                const int ci = r.drive ? jm : s, cj = r.drive ? s : jm;
                int i0, j0, d0i, d0j, c0i, c0j;
                const int mq = fold_canon(ci, cj, nh, n1, i0, j0);
                fold_step(mq, si, sj, d0i, d0j);
                fold_step(mq, mi, mj, c0i, c0j);
                for (int t = (mq - m) & 3; t > 0; --t) {
                    fold_rot_up(accB[0]); fold_rot_up(accB[1]);
                    if (F == 2) { fold_rot_dn(accT[0]); fold_rot_dn(accT[1]); }
                }
                m = mq;
                int offB = (i0 + PAD_M) * P.fis + (j0 + PAD_M) * P.fjs + kk, offT = (j0 + PAD_M) * P.fis + (i0 + PAD_M) * P.fjs + kk;
                const int drowB = d0i * P.fis + d0j * P.fjs, drowT = d0j * P.fis + d0i * P.fjs;
                const int dcolB = c0i * P.fis + c0j * P.fjs, dcolT = c0j * P.fis + c0i * P.fjs;
                const int seg_end = s < nh ? min(nh, s_hi) : s_hi;
                bool mixed = false;
                constexpr bool DEFER = FOLD_DEFER && F == 2;
                int pB = 0, pT = 0;
                float pw = 0.0f;                                     // the noted z-neighbour cell of this lane and its weight (0: none)
                auto flush = [&]() {
                    if (pw > 0.0f) {
                        CBCT_DEV_ASSERT(pB >= 0 && pB < P.stage_cells && (F == 1 || (pT >= 0 && pT < P.stage_cells)));
                        fold_fma(accB[0], pw, __ldg(fold + pB)); fold_fma(accB[1], pw, __ldg(fold_hi + pB));
                        if (F == 2) { fold_fma(accT[0], pw, __ldg(fold + pT)); fold_fma(accT[1], pw, __ldg(fold_hi + pT)); }
                        pw = 0.0f;
                    }
                };
                for (; s < seg_end; ++s) {
                    const float sy = __saturatef((nexty - y0) * r.inv_m);
                    const float sz = __saturatef((nextz - z0) * rz.inv_mz);
                    const bool cy = sy < 1.0f, cz = sz < 1.0f;
                    if (cy && nexty == 0.0f) { mixed = true; break; }      // crosses the centre plane of the minor axis
                    if (DEFER && !cy) {
                        // No in-plane crossing in this slab -- the same for every lane of the warp.  The first cell takes sz (1
                        // unless the lane crosses a z-plane here); the z-neighbour's share 1 - sz is owed by the few lanes that do
                        // cross.  The walk is bound by the bytes its loads REQUEST (a 16-byte load costs the LSU four passes however
                        // many lanes are predicated off), so that cell is not fetched now: the lane notes its offset and weight, and
                        // the warp fetches all noted cells at once when a lane must note a second one (and at the end of the run).
                        const bool ov = cz && pw > 0.0f;
                        if (__any_sync(__activemask(), ov)) flush();
                        CBCT_DEV_ASSERT(offB >= 0 && offB < P.stage_cells && (F == 1 || (offT >= 0 && offT < P.stage_cells)));
                        const float4 a0 = __ldg(fold + offB), a1 = __ldg(fold_hi + offB);
                        float4 ta0, ta1;
                        if (F == 2) { ta0 = __ldg(fold + offT); ta1 = __ldg(fold_hi + offT); }
                        const int zc = cz ? dk : 0;
                        if (cz) { pB = offB + dk; pT = offT + dk; pw = 1.0f - sz; }
                        fold_fma(accB[0], sz, a0); fold_fma(accB[1], sz, a1);
                        if (F == 2) { fold_fma(accT[0], sz, ta0); fold_fma(accT[1], sz, ta1); }
                        offB += zc + drowB; offT += zc + drowT;
                        if (cz) nextz += sgnz;
                        d += 1.0f;
                        y0 = fmaf(d, r.m, r.a0);
                        z0 = fmaf(d, rz.mz, rz.za);
                        continue;
                    }
                    const float lo = fminf(sy, sz);
                    const float hi = (cy && cz) ? fmaxf(sy, sz) : lo;
                    const float wl = 1.0f - hi;
                    const int zc = cz ? dk : 0;
                    const int offcB = offB + (cy ? dcolB : 0) + zc, offcT = offT + (cy ? dcolT : 0) + zc;
                    CBCT_DEV_ASSERT(offB >= 0 && offB < P.stage_cells && offcB >= 0 && offcB < P.stage_cells);
                    CBCT_DEV_ASSERT(F == 1 || (offT >= 0 && offT < P.stage_cells && offcT >= 0 && offcT < P.stage_cells));
                    const float4 a0 = __ldg(fold + offB), a1 = __ldg(fold_hi + offB), c0 = __ldg(fold + offcB), c1 = __ldg(fold_hi + offcB);
                    float4 ta0, ta1, tc0, tc1;
                    if (F == 2) {
                        ta0 = __ldg(fold + offT); ta1 = __ldg(fold_hi + offT); tc0 = __ldg(fold + offcT); tc1 = __ldg(fold_hi + offcT);
                    }
                    fold_fma(accB[0], lo, a0); fold_fma(accB[0], wl, c0);
                    fold_fma(accB[1], lo, a1); fold_fma(accB[1], wl, c1);
                    if (F == 2) {
                        fold_fma(accT[0], lo, ta0); fold_fma(accT[0], wl, tc0);
                        fold_fma(accT[1], lo, ta1); fold_fma(accT[1], wl, tc1);
                    }
                    if (hi > lo) {      // a third cell (rare): the in-plane neighbour lies in the same quadrant here
                        const float wm = hi - lo;
                        const bool yfirst = sy < sz;
                        const int oB = offB + (yfirst ? dcolB : dk);
                        CBCT_DEV_ASSERT(oB >= 0 && oB < P.stage_cells);
                        fold_fma(accB[0], wm, __ldg(fold + oB)); fold_fma(accB[1], wm, __ldg(fold_hi + oB));
                        if (F == 2) {
                            const int oT = offT + (yfirst ? dcolT : dk);
                            CBCT_DEV_ASSERT(oT >= 0 && oT < P.stage_cells);
                            fold_fma(accT[0], wm, __ldg(fold + oT)); fold_fma(accT[1], wm, __ldg(fold_hi + oT));
                        }
                    }
                    offB = offcB + drowB; offT = offcT + drowT;
                    if (cy) nexty += sgny;
                    if (cz) nextz += sgnz;
                    d += 1.0f;
                    y0 = fmaf(d, r.m, r.a0);
                    z0 = fmaf(d, rz.mz, rz.za);
                }
                if (DEFER) flush();                                  // before the frame of the sums changes
                if (mixed) {
                    // ---- the slab that crosses the minor axis' centre plane: its cells lie in two quadrants ----
                    const float sy = __saturatef((nexty - y0) * r.inv_m);
                    const float sz = __saturatef((nextz - z0) * rz.inv_mz);
                    const bool cz = sz < 1.0f;                              // cy holds
                    const float lo = fminf(sy, sz);
                    const float hi = cz ? fmaxf(sy, sz) : lo;
                    const float wl = 1.0f - hi;
                    const int zc = cz ? dk : 0;
                    const int jx = (int)nexty - (posy ? 1 : 0) + nh, kx = (int)nextz - (posz ? 1 : 0) + P.cz + PAD_Z;
                    const int xi = r.drive ? jx : s, xj = r.drive ? s : jx;
                    fold_cell<F>(P, fold, xi, xj, kx, lo, m, accB, accT);
                    fold_cell<F>(P, fold, xi + mi, xj + mj, kx + zc, wl, m, accB, accT);
                    if (hi > lo) {
                        const bool yfirst = sy < sz;
                        fold_cell<F>(P, fold, xi + (yfirst ? mi : 0), xj + (yfirst ? mj : 0), kx + (yfirst ? 0 : dk), hi - lo, m, accB, accT);
                    }
                    nexty += sgny;
                    if (cz) nextz += sgnz;
                    d += 1.0f;
                    y0 = fmaf(d, r.m, r.a0);
                    z0 = fmaf(d, rz.mz, rz.za);
                    ++s;
                }
            }
        }
        for (int t = (4 - m) & 3; t > 0; --t) {                // back to the frame of quadrant 0: component c = quarter turn c
            fold_rot_up(accB[0]); fold_rot_up(accB[1]);
            if (F == 2) { fold_rot_dn(accT[0]); fold_rot_dn(accT[1]); }
        }
        float acc[4 * F * 2];
#pragma unroll
        for (int mm = 0; mm < 2; ++mm)
#pragma unroll
            for (int q = 0; q < 4; ++q) {
                acc[mm * 4 * F + q] = accB[mm][q];
                if (F == 2) acc[mm * 4 * F + 4 + q] = accT[mm][(3 - q) & 3];
            }
        forward_epilogue<4, 2, MODE, F>(P, r, v, acc, a, ar, iu, iv, y, out, sq);
    }
    if (MODE == 1 || MODE == 4) {
        double s[1];
        s[0] = block_sum(sq, slot);
        if (counter) publish_and_finalize<1>(s, 1, partials, stride, counter, sum_out, slot);
        else publish_only<1>(s, 1, partials, stride, ((unsigned)blockIdx.z * (F == 2 ? P.npairs : P.nbase) + a) * gridDim.x + blockIdx.x);
    }
}

constexpr int FWD_BX = 32, FWD_BY = 8;      // count_samples_kernel block

// S = number of (ray, voxel) pairs with positive length, by the same slab decomposition with the
// cell taken from floor() and tested against the true volume bounds.  Not on the hot path.
__global__ void __launch_bounds__(FWD_BX *FWD_BY)
count_samples_kernel(const LevelParams P, const RayU *__restrict__ rayu, double *__restrict__ partials)
{
    __shared__ double slot[32];
    const int iu = blockIdx.x * FWD_BX + threadIdx.x;
    const int iv = blockIdx.y * FWD_BY + threadIdx.y;
    const int a = blockIdx.z;
    int cnt = 0;
    if (iu < P.nu && iv < P.nv) {
        const RayU r = load_rayu(rayu, a * P.nu + iu);
        const float v = fmaf((float)iv, P.dv, P.v0);
        const RayZ rz = ray_z(r, v, P.sz);
        const int nd = r.drive ? P.ny : P.nx, nm = r.drive ? P.nx : P.ny;
        const int cd = r.drive ? P.cy : P.cx, cm = r.drive ? P.cx : P.cy;
        for (int s = 0; s < nd; ++s) {
            const float d0 = (float)(s - cd), d1 = (float)(s + 1 - cd);
            const float y0 = fmaf(d0, r.m, r.a0), z0 = fmaf(d0, rz.mz, rz.za);
            const float y1 = fmaf(d1, r.m, r.a0), z1 = fmaf(d1, rz.mz, rz.za);
            const float fy0 = floorf(y0), fy1 = floorf(y1), fz0 = floorf(z0), fz1 = floorf(z1);
            float sy = 1.0f, sz = 1.0f;
            if (fy0 != fy1) sy = __saturatef((fmaxf(fy0, fy1) - y0) * r.inv_m);
            if (fz0 != fz1) sz = __saturatef((fmaxf(fz0, fz1) - z0) * rz.inv_mz);
            const float wa = fminf(sy, sz), wb = fmaxf(sy, sz) - wa, wc = 1.0f - fmaxf(sy, sz);
            const int j0 = (int)fy0 + cm, j1 = (int)fy1 + cm, k0 = (int)fz0 + P.cz, k1 = (int)fz1 + P.cz;
            if (wa > 0.0f && (unsigned)j0 < (unsigned)nm && (unsigned)k0 < (unsigned)P.nz) ++cnt;
            if (wb > 0.0f) {
                const int jb = sy < sz ? j1 : j0, kb = sy < sz ? k0 : k1;
                if ((unsigned)jb < (unsigned)nm && (unsigned)kb < (unsigned)P.nz) ++cnt;
            }
            if (wc > 0.0f && (unsigned)j1 < (unsigned)nm && (unsigned)k1 < (unsigned)P.nz) ++cnt;
        }
    }
    double s = block_sum((double)cnt, slot);
    if (threadIdx.x == 0 && threadIdx.y == 0)
        partials[((size_t)blockIdx.z * gridDim.y + blockIdx.y) * gridDim.x + blockIdx.x] = s;
}

template <int R, int M, int F>
static void launch_forward_mode(const cbct_geometry *g, const LevelParams &P, dim3 gr, dim3 b, cudaStream_t st, int mode,
                                const void *stage, const RayU *rayu, const float *d_y, float *d_out, double *d_sum_sq,
                                int a_off, bool fused_sum)
{
    unsigned int *ctr = fused_sum ? g->d_counter : nullptr;
    if (mode == 0) forward_kernel<R, M, 0, F><<<gr, b, 0, st>>>(P, stage, rayu, nullptr, d_out, nullptr, 0, nullptr, nullptr, a_off);
    else if (mode == 2) forward_kernel<R, M, 2, F><<<gr, b, 0, st>>>(P, stage, rayu, nullptr, d_out, nullptr, 0, nullptr, nullptr, a_off);
    else if (mode == 4) forward_kernel<R, M, 4, F><<<gr, b, 0, st>>>(P, stage, rayu, d_y, d_out, g->d_partials, g->partials_stride,
                                                                    ctr, d_sum_sq, a_off);
    else forward_kernel<R, M, 1, F><<<gr, b, 0, st>>>(P, stage, rayu, d_y, d_out, g->d_partials, g->partials_stride,
                                                      ctr, d_sum_sq, a_off);
}

template <int F>
static void launch_forward_fold_mode(const cbct_geometry *g, const LevelParams &P, dim3 gr, dim3 b, cudaStream_t st, int mode,
                                     const void *stage, const RayU *rayu, const float *d_y, float *d_out, double *d_sum_sq,
                                     int a_off, bool fused_sum)
{
    unsigned int *ctr = fused_sum ? g->d_counter : nullptr;
    const float4 *fold = reinterpret_cast<const float4 *>(stage);
    if (mode == 0) forward_fold_kernel<0, F><<<gr, b, 0, st>>>(P, fold, rayu, nullptr, d_out, nullptr, 0, nullptr, nullptr, a_off);
    else if (mode == 2) forward_fold_kernel<2, F><<<gr, b, 0, st>>>(P, fold, rayu, nullptr, d_out, nullptr, 0, nullptr, nullptr, a_off);
    else if (mode == 4) forward_fold_kernel<4, F><<<gr, b, 0, st>>>(P, fold, rayu, d_y, d_out, g->d_partials, g->partials_stride,
                                                                  ctr, d_sum_sq, a_off);
    else forward_fold_kernel<1, F><<<gr, b, 0, st>>>(P, fold, rayu, d_y, d_out, g->d_partials, g->partials_stride,
                                                   ctr, d_sum_sq, a_off);
}

// units of a forward launch (its grid's y dimension, and what a sharded launch splits): base views, or view pairs
int forward_units(const Level &L) { return (L.p.nsym == 4 && L.p.nmir == 2 && L.p.nrefl == 2) ? L.p.npairs : L.p.nbase; }

cbct_status launch_forward(const cbct_geometry *g, const Level &L, const float *d_vol, const float *d_y,
                           float *d_out, int mode, double *d_sum_sq, cudaStream_t st, const Shard *sh)
{
    const LevelParams &P = L.p;
    if (sh && mode != 1 && mode != 2) return cbct_fail(CBCT_ERR_INVALID_ARG, "launch_forward: a sharded launch writes the residual stack");
    dim3 b(FWD_BX, FWD_BY);
    if (mode == 3) {
        dim3 gr((P.nu + FWD_BX - 1) / FWD_BX, (P.nv + FWD_BY - 1) / FWD_BY, P.np);
        const size_t nblk = (size_t)gr.x * gr.y * gr.z;
        if (nblk > (size_t)g->partials_stride) return cbct_fail(CBCT_ERR_INVALID_ARG, "projection stack too large for the reduction buffer");
        count_samples_kernel<<<gr, b, 0, st>>>(P, L.d_rayu, g->d_partials);
        CBCT_LAUNCH_CHECK(g);
        finalize_sums_kernel<<<1, 256, 0, st>>>(g->d_partials, (int)nblk, 1, g->partials_stride, d_sum_sq);
        CBCT_LAUNCH_CHECK(g);
        return CBCT_OK;
    }
    {
        StageTimer t(g, st, ST_TRANSPOSE);
        dim3 tb(32, 8);
        if (P.fold) {
            dim3 tg((P.nhP + FOLD_T - 1) / FOLD_T, (P.nhP + FOLD_T - 1) / FOLD_T, 2 * ((P.nzP + FOLD_K - 1) / FOLD_K));
            stage_volume_fold_kernel<<<tg, 256, 0, st>>>(d_vol, reinterpret_cast<float4 *>(L.d_stage), P.nx, P.nz, P.nhP, P.nzP);
        } else if (P.nmir == 2) {
            if (P.nx % 4 == 0 && P.nzP % 2 == 0 && (uintptr_t)d_vol % 16 == 0) {
                dim3 tg((P.nx + STG_I - 1) / STG_I, (P.nzP + STG_K - 1) / STG_K, P.ny);
                stage_volume_packed_vec_kernel<<<tg, 256, 0, st>>>(d_vol, reinterpret_cast<float4 *>(L.d_stage), P.nx, P.ny, P.nz,
                                                                    P.istride, P.jstride);
            } else {
                dim3 tg((P.nx + 31) / 32, (P.nzP + 31) / 32, P.ny);
                stage_volume_packed_kernel<<<tg, tb, 0, st>>>(d_vol, reinterpret_cast<float2 *>(L.d_stage), P.nx, P.ny, P.nz,
                                                             P.istride, P.jstride);
            }
        } else {
            dim3 tg((P.nx + 31) / 32, (P.nz + 31) / 32, P.ny);
            stage_volume_kernel<<<tg, tb, 0, st>>>(d_vol, L.d_stage, P.nx, P.ny, P.nz, P.istride, P.jstride);
        }
        CBCT_LAUNCH_CHECK(g);
    }
    const int bu = P.fold ? FOLD_BU : FWD_BU;
    b = dim3(FWD_BV, bu);
    const int units = forward_units(L);          // base views, or view pairs where the walk also serves the reflected rays
    dim3 gr((P.nu + bu - 1) / bu, units, (P.nv / P.nmir + FWD_BV - 1) / FWD_BV);
    const size_t nblk = (size_t)gr.x * gr.y * gr.z;             // of the full launch: the numbering of the partial sums
    if ((mode == 1 || mode == 4) && nblk > (size_t)g->partials_stride)
        return cbct_fail(CBCT_ERR_INVALID_ARG, "projection stack too large for the reduction buffer");
    int a_off = 0;
    if (sh) {
        if (sh->base_lo < 0 || sh->base_hi > units || sh->base_lo > sh->base_hi) return cbct_fail(CBCT_ERR_INVALID_ARG, "launch_forward: bad shard");
        a_off = sh->base_lo;
        gr.y = sh->base_hi - sh->base_lo;
        if (gr.y == 0) return CBCT_OK;
    }
    {
        StageTimer t(g, st, ST_FORWARD);
        const bool fused = sh == nullptr;
        if (P.fold && P.nrefl == 2) launch_forward_fold_mode<2>(g, P, gr, b, st, mode, L.d_stage, L.d_rayu, d_y, d_out, d_sum_sq, a_off, fused);
        else if (P.fold) launch_forward_fold_mode<1>(g, P, gr, b, st, mode, L.d_stage, L.d_rayu, d_y, d_out, d_sum_sq, a_off, fused);
        else if (P.nsym == 4 && P.nmir == 2 && P.nrefl == 2) launch_forward_mode<4, 2, 2>(g, P, gr, b, st, mode, L.d_stage, L.d_rayu, d_y, d_out, d_sum_sq, a_off, fused);
        else if (P.nsym == 4 && P.nmir == 2) launch_forward_mode<4, 2, 1>(g, P, gr, b, st, mode, L.d_stage, L.d_rayu, d_y, d_out, d_sum_sq, a_off, fused);
        else if (P.nsym == 4) launch_forward_mode<4, 1, 1>(g, P, gr, b, st, mode, L.d_stage, L.d_rayu, d_y, d_out, d_sum_sq, a_off, fused);
        else if (P.nmir == 2) launch_forward_mode<1, 2, 1>(g, P, gr, b, st, mode, L.d_stage, L.d_rayu, d_y, d_out, d_sum_sq, a_off, fused);
        else launch_forward_mode<1, 1, 1>(g, P, gr, b, st, mode, L.d_stage, L.d_rayu, d_y, d_out, d_sum_sq, a_off, fused);
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
