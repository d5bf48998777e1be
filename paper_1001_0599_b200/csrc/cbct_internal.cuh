// cbct_internal.cuh -- shared declarations of the CUDA product path (libcbct).
// Nothing here is used by, or uses, the CPU oracle under oracle/.
#pragma once
#include <cuda.h>
#include <cuda_runtime.h>
#include <stdint.h>
#include <vector>
#include "../../include/cbct.h"

// One entry per (view, detector column iu): everything about the ray fan of that column
// that does not depend on the detector row.  Computed in fp64 on the host at create
// (Eq. 1, L374 Eq. A2), rounded once to fp32, and read by BOTH projectors so
// that P and P^T evaluate bit-identical ray positions.
//
// "Index coordinates": axis a measured in voxels from grid plane n_a/2 (integer division),
// so voxel i spans [i - n/2, i + 1 - n/2) and grid planes sit on integers.
// The ray is driven along x when it crosses at least as many x-planes as y-planes
// (drive = 0: slab = x index, in-plane minor axis = y), else along y (drive = 1).
// Along the driving coordinate D (index units):
//     minor(D) = a0 + D * m,        |m| <= 1
//     z(D)     = sz + v * q * (D - sd)        (v = detector row coordinate in mm)
//     length of the ray inside one slab (mm) = L(u,v) * inv_dd,  L = sqrt(c_l + v^2)
struct __align__(16) RayU {
    float a0, m, inv_m, q;
    float sd, inv_dd, c_l;
    int drive;
};

// Per-view constants of the voxel -> detector map (Eq. A6) used by the
// back-projector to bound the set of rays that can cross a voxel.
struct __align__(16) ViewC {
    float c, s;        // cos, sin of the view angle
    float dn, du;      // half extents of a voxel along e_n and e_u (mm), slightly inflated
};

// Padding (voxels) of the staged volume copies on the minor in-plane axis and on z: the forward
// projector walks a ray only through slabs where it is within half a voxel of the volume, so
// every cell it can touch -- including the one-cell slack of its incremental cell tracking
// -- lies inside the zero-filled margin and no load needs a bounds test.
constexpr int PAD_M = 4, PAD_Z = 4;

struct LevelParams {
    int nx, ny, nz, nu, nv, np;
    int nsym, nbase;           // views handled per thread by rotation symmetry (1 or 4); np / nsym
    int nmir;                  // 2 when the z-mirror image of every ray / voxel shares its weights, else 1
    int nrefl, npairs;         // 2 when the view set is also symmetric under theta -> -theta (forward.cu walks view pairs:
                               // npairs = nbase / 2 + 1 units), else 1
    int stage_cells, t_entries; // cells of the staged copy / entries (R floats) of the residual stack: bounds of the gathers
    int tP, tXP;               // residual stack: rows of a detector column stored in tP planes by row % tP (1 = plain), tXP = nv / tP
                               // entries each: row iv sits at (iv % tP) * tXP + iv / tP of its column (back_tma.cu)
    int nyP, nzP;              // padded extents of the staged volume [i + PM][j + PM][k + PZ] (k fastest)
    int istride, jstride;      // its element strides along i and j (nyP * nzP, nzP)
    int fold, nhP, fis, fjs;   // fold != 0: the staged copy is folded onto the first quadrant (forward.cu): [i0 + PM][j0 + PM][kk]
                               // entries of 8 floats, nhP = nx / 2 + PM canonical cells per axis, entry strides fis = nhP * nzP, fjs = nzP
    int cx, cy, cz;            // n/2 (integer): index of the grid plane at index coordinate 0
    float hx, hy, hz;
    float x0, y0, z0;          // centre of voxel 0 in mm
    float u0, du, v0, dv;      // centre of pixel 0 and pitch in mm
    float inv_du, inv_dv;
    float sz;                  // source z in index coordinates
    float sad, sdd;
    int bc_xy, bc_z;
};

// ---- back_tma.cu: the TMA / shared-memory back-projector's per-level plan ----
constexpr int BT_MAXC = 8;      // candidate detector columns per (voxel column, base view, image)
constexpr int BT_NST = 2;       // depth of the tile ring
constexpr int BT_NMAPS = 5;     // tensor maps with boxes of 1, 2, 4, 8, 16 detector columns
struct BtMaps { CUtensorMap m[BT_NMAPS]; };
struct BtParams {
    int XB;                     // entries (rows) per plane of a tile column; a multiple of 8
    int ncols;                  // tile columns: the widest brick shadow of the level
    int plane_bytes, half_bytes, stage_bytes;   // ncols * XB * 16; x tP (the rows of one volume half); x 2
    int list_off, view_off, hdr_off, bar_off, total;   // shared-memory carve-up (bytes)
    int nzh;                    // nz / 2
    int vec4;                   // results may leave with 16-byte stores
    int zu_fast;                // launch order: the z-units of a brick next to one another (else the z-unit is the slowest index)
    float ic_scale;             // hz * sdd / dv: detector rows per z-index at unit depth
    float c0v_m;                // -v0 / dv - 2e-3: row index of v = 0, minus the range tolerance
};
struct BtConsts { float c0v_m, dv, v0; int rr_max, plane_step8, step_even, step_odd, KB; };
struct BtPlan {
    bool ok = false;
    int BI = 0, BJ = 0, CPW = 0, NSLOT = 0, TP = 1, minb = 1, ZV = 1;    // ZV: voxels per lane along z (blocks of 32 ZV slices)
    BtParams q;
    BtMaps maps;
    int4 *d_hdrs = nullptr;     // stage headers of every (z-unit, brick), 4 n_base int4 each (with d_lists)
    float4 *d_lists = nullptr;  // in-plane lists of every (first-quadrant voxel column, base view), 32 float4 each; NULL: on the fly
};

struct Level {
    LevelParams p;
    BtPlan bt;
    double hx, hy, hz, du, dv;
    size_t nvox, nray;
    RayU *d_rayu = nullptr;     // [np][nu]
    ViewC *d_view = nullptr;    // [np]
    double2 *d_cs = nullptr;    // [np] cos, sin of the view angles in fp64 (back_eq6.cu)
    // scratch (all fp32 unless noted)
    float *d_stage = nullptr;   // zero-padded, z-fastest copy of the volume: [i+PM][j+PM][k+PZ]
    size_t stage_elems = 0;
    float *d_T = nullptr;       // residual scaled by L(u,v): what P^T consumes; detector rows fastest:
                                // [np][nu][nv], or [nbase][nu][nv][4] (the four quarter-turn views
                                // interleaved) when nsym == 4
    float *d_g = nullptr;       // g of Algorithm A1
    float *d_d = nullptr;       // descent direction of the ROF sub-solver
    float *d_f2 = nullptr;      // second volume (ping-pong / level volume)
    float *d_f = nullptr;       // level volume for levels > 0 and for the host entry point
    float *d_prev = nullptr;    // the volume that entered the current iteration (convergence test, NEXT-2)
    float *d_y = nullptr;       // binned data for levels > 0; staging for level 0 host entry
    int back_maxc = 1 << 30;    // upper bound of the detector columns in the shadow of one voxel's (i,j) square (back.cu)
    mutable double lhat = -1.0; // A5 step bound: a property of the geometry alone, computed on first use
};

struct cbct_geometry {
    cbct_geometry_desc desc;
    std::vector<double> angles;
    std::vector<Level> levels;
    double *d_partials = nullptr;   // fp64 block partials, 4 rows of partials_stride
    int partials_stride = 0;        // >= the block count of every reducing kernel on every level
    double *d_scalars = nullptr;    // reduced scalars on the device
    unsigned int *d_counter = nullptr;  // ticket of the fused reductions (reduce.cuh); 0 between kernels
    double *h_scalars = nullptr;    // pinned host mirror
    double *d_objective = nullptr;  // per-iteration E1, E2 pairs
    int objective_cap = 0;
    unsigned long long device_bytes = 0;
    mutable unsigned long long launches = 0;
    int allow_symmetry = 1;
    int stage_timing = 0;
    mutable float stage_ms[CBCT_N_STAGES] = {0};
    mutable unsigned long long stage_calls[CBCT_N_STAGES] = {0};
    cudaEvent_t ev[5] = {nullptr, nullptr, nullptr, nullptr, nullptr};   // 0,1 whole call; 2,3 stage timers; 4 first TV trial
    int sm_count = 148;
    int disable_tma = 0;            // cbct_geometry_desc::kernel_flags bit 0
    int host_armijo = 0;            // bit 1: the host-sequenced Armijo loop instead of the cooperative TV-prox kernel
    int tv_scalar_tiles = 0;        // bit 2: the TV passes on the 32-voxel warp tiles only
    int no_fold = 0;                // bit 5: the forward projector never reads the folded staged copy
    int no_reflection = 0;          // bit 4: the forward projector walks base views, never view pairs
    int back_lists_on_the_fly = 0;  // bit 3: the TMA back-projector works its in-plane lists out itself (no table at create)
    unsigned int *d_errflag = nullptr;  // device-side "a create-time bound did not hold" counter (back_tma.cu); 0 always
};

// Debug builds (-DCBCT_ASSERT): device-side bounds checks of every gather index (compute-sanitizer stand-in).
#ifdef CBCT_ASSERT
#include <assert.h>
#define CBCT_DEV_ASSERT(x) assert(x)
#else
#define CBCT_DEV_ASSERT(x) ((void)0)
#endif

constexpr int kScalars = 24;     // 0-2 gradient-pass sums, 4-5 trial sums, 8 E1, 9 Lhat max, 10 S, 16-21 cooperative TV-prox report

// Attribution of device time to one kernel (or a short fixed group): CUDA events around the
// launches on the library's stream, only when cbct_set_stage_timing switched it on (it adds a
// synchronisation per stage, so whole-call timings are taken with it off).
enum { ST_TRANSPOSE = 0, ST_FORWARD, ST_BACK, ST_TV_GRAD, ST_TV_TRIAL, ST_TV_UPDATE, ST_REDUCE, ST_TRANSFER };
struct StageTimer {
    const cbct_geometry *g;
    cudaStream_t st;
    int slot;
    bool on;
    StageTimer(const cbct_geometry *g_, cudaStream_t st_, int slot_) : g(g_), st(st_), slot(slot_), on(g_->stage_timing != 0)
    {
        if (on) cudaEventRecord(g->ev[2], st);
    }
    ~StageTimer()
    {
        if (!on) return;
        cudaEventRecord(g->ev[3], st);
        cudaEventSynchronize(g->ev[3]);
        float ms = 0.f;
        cudaEventElapsedTime(&ms, g->ev[2], g->ev[3]);
        g->stage_ms[slot] += ms;
        g->stage_calls[slot] += 1;
    }
};

// error plumbing (geometry.cu)
cbct_status cbct_fail(cbct_status st, const char *fmt, ...);
#define CBCT_CUDA(expr)                                                                         \
    do {                                                                                        \
        cudaError_t e__ = (expr);                                                               \
        if (e__ != cudaSuccess)                                                                 \
            return cbct_fail(e__ == cudaErrorMemoryAllocation ? CBCT_ERR_OOM : CBCT_ERR_CUDA,   \
                             "%s: %s", #expr, cudaGetErrorString(e__));                         \
    } while (0)
#define CBCT_LAUNCH_CHECK(g)                                                                    \
    do {                                                                                        \
        (g)->launches++;                                                                        \
        cudaError_t e__ = cudaGetLastError();                                                   \
        if (e__ != cudaSuccess)                                                                 \
            return cbct_fail(CBCT_ERR_CUDA, "kernel launch: %s", cudaGetErrorString(e__));      \
    } while (0)

static inline const Level *get_level(const cbct_geometry *g, int level)
{
    if (!g || level < 0 || level >= (int)g->levels.size()) return nullptr;
    return &g->levels[level];
}

// A rank's share of the two projectors in a sharded reconstruction (fbs.cu): base views [base_lo, base_hi) of the forward
// projector, z-units [zu_lo, zu_hi) of the back-projector (back_zunit() slices of the lower half volume each -- of the whole
// volume without mirror symmetry -- with their mirror images).  NULL = everything, with the fused reduction.
struct Shard {
    int base_lo, base_hi, zu_lo, zu_hi;
};
int forward_units(const Level &L);
int back_zunit(const Level &L);
int back_nzunits(const Level &L);

// internal launchers (asynchronous on `st`)
// forward.cu : mode 0: out = P vol (plain layout).
//              mode 1: out = L * (P vol - y) in the d_T layout, *d_sum_sq = sum (P vol - y)^2.
//              mode 2: out = L * (P vol) in the d_T layout.
//              mode 3: *d_sum_sq = number of (ray, voxel) pairs, no volume read
//              mode 4: out = P vol - y (plain layout), *d_sum_sq = sum (P vol - y)^2
//              With a shard (modes 1, 2): only its base views; mode 1 then leaves the blocks' partial sums of (P vol - y)^2
//              in g->d_partials row 0 at their index in the full launch (no sum is formed).
cbct_status launch_forward(const cbct_geometry *g, const Level &L, const float *d_vol, const float *d_y,
                           float *d_out, int mode, double *d_sum_sq, cudaStream_t st, const Shard *sh = nullptr);
// back.cu : scaled != 0: d_in already holds L*T in the d_T layout; else plain layout, unscaled.
//           out = f - coef * P^T in (f may be NULL: out = P^T in)
//           With a shard: only the voxels of its z-units are written.
cbct_status launch_back(const cbct_geometry *g, const Level &L, const float *d_in, int scaled,
                        const float *d_f, float coef, float *d_out, cudaStream_t st, const Shard *sh = nullptr);
// back_tma.cu : plan of the TMA back-projector for a level (create time; needs L.d_T), and its launch (input = L.d_T)
cbct_status bt_plan_level(const cbct_geometry *g, Level &L);
cbct_status launch_back_tma(const cbct_geometry *g, const Level &L, const float *d_f, float coef, float *d_out, cudaStream_t st,
                            const Shard *sh = nullptr);
// back_eq6.cu : out = f - coef * b6(T) with T in the plain [view][row][column] layout (f may be NULL: out = b6(T))
cbct_status launch_back_eq6(const cbct_geometry *g, const Level &L, const float *d_T, const float *d_f, float coef,
                            float *d_out, cudaStream_t st);
// metrics.cu : *sum_d2 = sum (a - b)^2, *sum_b2 = sum b^2 over n elements (fp64, fixed order); synchronises the stream
cbct_status volume_change(const cbct_geometry *g, size_t n, const float *d_a, const float *d_b, double *sum_d2,
                          double *sum_b2, cudaStream_t st);
// tv.cu
// `ahead` (may be NULL): work the caller wants queued behind the first trial pass, which has left the candidate result in
// d_f; it is called once, before the host waits for that trial's sums.  *ahead_valid tells whether d_f still held that
// candidate when the call returned (the first step was accepted and was the last), i.e. whether the queued work is good.
struct TvAhead {
    cbct_status (*fn)(void *ctx);
    void *ctx;
    bool valid;
};
cbct_status run_tv_prox(const cbct_geometry *g, const Level &L, const float *d_g, float *d_f, double w,
                        int nonneg, const cbct_tv_params &tp, cbct_tv_report *rep, bool sync_report,
                        cudaStream_t st, TvAhead *ahead = nullptr);
cbct_status launch_tv_energy(const cbct_geometry *g, const Level &L, const float *d_f, double delta,
                             double *d_out, cudaStream_t st);
// transfer.cu
cbct_status launch_restrict(const cbct_geometry *g, const Level &fine, const float *d_fine, float *d_coarse, cudaStream_t st);
cbct_status launch_bin(const cbct_geometry *g, const Level &fine, const float *d_fine, float *d_coarse, cudaStream_t st);
cbct_status launch_prolong(const cbct_geometry *g, const Level &fine, const float *d_coarse, float *d_fine, cudaStream_t st);
cbct_status launch_max(const cbct_geometry *g, const float *d_x, size_t n, double *d_out, cudaStream_t st);
cbct_status launch_fill(const cbct_geometry *g, float *d_x, size_t n, float val, cudaStream_t st);
