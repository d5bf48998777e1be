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
    if (MODE == 1 || MODE == 4) {        // E2 numerator: sum of squared residuals, second stage fused (reduce.cuh)
        double s[1];
        s[0] = block_sum(sq, slot);
        if (counter) publish_and_finalize<1>(s, 1, partials, stride, counter, sum_out, slot);
        else publish_only<1>(s, 1, partials, stride, ((unsigned)blockIdx.z * (F == 2 ? P.npairs : P.nbase) + a) * gridDim.x + blockIdx.x);   // sharded launch
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
        if (P.nmir == 2) {
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
    b = dim3(FWD_BV, FWD_BU);
    const int units = forward_units(L);          // base views, or view pairs where the walk also serves the reflected rays
    dim3 gr((P.nu + FWD_BU - 1) / FWD_BU, units, (P.nv / P.nmir + FWD_BV - 1) / FWD_BV);
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
        if (P.nsym == 4 && P.nmir == 2 && P.nrefl == 2) launch_forward_mode<4, 2, 2>(g, P, gr, b, st, mode, L.d_stage, L.d_rayu, d_y, d_out, d_sum_sq, a_off, fused);
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
