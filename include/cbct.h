/*
 * cbct.h -- C ABI of libcbct: the forward-backward-splitting (FBS) hot path of
 * Jia et al., "GPU-based Fast Low-dose Cone Beam CT Reconstruction via Total
 * Variation" (arxiv 1001.0599), hand-written CUDA for sm_100a (NVIDIA B200), one GPU.
 *
 * Citations are PAPER.md line numbers (L..) with the equation / section they fall in;
 * "reading S.." refers to the list of readings in DESIGN.md section 4.
 *
 * Conventions common to every call
 *   - Pointers named d_* are CALLER-OWNED DEVICE pointers (contiguous fp32), h_* are
 *     caller-owned HOST pointers.  The library never frees or reallocates them.
 *   - Volume layout  f[(k*ny + j)*nx + i]  (x fastest; z = rotation axis = superior-inferior).
 *     Projection layout  p[(a*nv + jv)*nu + iu]  (u fastest; a = view index).
 *   - `cuda_stream` is a cudaStream_t passed as void* (NULL = the legacy default stream).
 *     Operator calls are asynchronous on that stream; calls that fill a report
 *     synchronise the stream before returning.
 *   - The handle owns every scratch buffer (allocated at create; timed calls allocate
 *     nothing).  A handle is NOT thread-safe: one call at a time per handle.
 *   - Errors are return codes only; nothing throws or exits across the ABI.  After an
 *     error the outputs are unspecified.  cbct_last_error() gives a thread-local message.
 *   - Same binary + same inputs => bitwise identical outputs (no floating-point atomics,
 *     fixed launch shapes, fixed-order fp64 reductions).
 *   - There is no CPU fallback: without an sm_100 device create returns CBCT_ERR_UNSUPPORTED.
 */
#ifndef CBCT_H
#define CBCT_H

#ifdef __cplusplus
extern "C" {
#endif

typedef struct cbct_geometry cbct_geometry; /* opaque */

typedef enum {
    CBCT_OK = 0,
    CBCT_ERR_INVALID_ARG = 1, /* NULL pointer, non-positive size/pitch, bad level count ... */
    CBCT_ERR_GEOMETRY = 2,    /* sad >= sdd, volume reaches the source or the detector plane,
                                 a ray direction the driving-axis traversal cannot take */
    CBCT_ERR_CUDA = 3,        /* a CUDA runtime call failed (message in cbct_last_error) */
    CBCT_ERR_OOM = 4,         /* device allocation failed */
    CBCT_ERR_UNSUPPORTED = 5  /* no sm_100 device */
} cbct_status;

enum { CBCT_BC_ZERO = 0, CBCT_BC_REFLECT = 1 };

/* Circular cone-beam acquisition (L89-L93 Eq. 1, Fig. 1, Appendix A2, A6 L401):
 *   view angle t:  e_n = (cos t, sin t, 0), e_u = (sin t, -cos t, 0), e_v = (0,0,1),
 *   source S = -sad e_n, detector point P(u,v) = S + sdd e_n + u e_u + v e_v  (sdd = L0),
 *   voxel (i,j,k) centre  x_i = (i - (nx-1)/2) hx + vol_off[0]  (same for y, z),
 *   pixel centre          u_i = (i - (nu-1)/2) du + det_off_u   (same for v),
 *   one ray per pixel centre.  All lengths in mm, angles in radians. */
typedef struct {
    int nx, ny, nz;
    double hx, hy, hz;
    double vol_off[3];
    int nu, nv;
    double du, dv, det_off_u, det_off_v;
    double sad, sdd;
    int n_proj;
    const double *angles_rad; /* n_proj angles; NULL => 2*pi*a/n_proj (L251); copied at create */
    int bc_xy, bc_z;          /* TV boundary rule: CBCT_BC_ZERO / CBCT_BC_REFLECT; the paper uses
                                 ZERO in x,y and REFLECT in z (L161) */
    int max_levels;           /* multi-grid levels to provision (>= 1); level l has every volume and
                                 detector dimension divided by 2^l, so all must be divisible */
    int no_symmetry;          /* 0 (default): when the in-plane grid is square, centred and even-sized and
                                 the views come in quarter-turn quadruples (angles[a + n_proj/4] = angles[a]
                                 + pi/2), both projectors compute each weight once for the four quarter-turn
                                 images of a ray; when the volume is centred in z and the detector in v
                                 (even nz, nv) also for the mirror image z -> -z.
                                 1: always use the generic one-ray-at-a-time kernels. */
    int kernel_flags;         /* 0 (default): every level takes the fastest kernels its geometry allows.
                                 CBCT_KERNEL_NO_TMA: never the TMA / shared-memory back-projector (cbct_geometry_back_path);
                                 for A/B measurements and for keeping the other paths under test. */
} cbct_geometry_desc;
#define CBCT_KERNEL_NO_TMA 1
#define CBCT_KERNEL_HOST_ARMIJO 2 /* cbct_tv_prox sequenced by the host (one stream synchronisation per Armijo trial) instead
                                     of the single cooperative kernel that takes every accept / shrink / stop decision on
                                     the device; same passes, same decisions.  For A/B measurements and tests. */
#define CBCT_KERNEL_BACK_LISTS_ON_THE_FLY 8 /* the TMA back-projector works out the in-plane part of its (voxel column, detector
                                              column) pairs at the start of every base view instead of reading the table
                                              cbct_geometry_create builds once (512 bytes per first-quadrant voxel column and
                                              base view); same bits either way.  For A/B measurements and tests. */
#define CBCT_KERNEL_NO_REFLECTION 16 /* the forward projector walks one base view per thread group even where the view set is
                                        also symmetric under theta -> -theta (then it walks view pairs: 16 rays per weight
                                        instead of 8).  For A/B measurements and tests. */
#define CBCT_KERNEL_NO_FOLD 32 /* the forward projector of a quarter-turn + mirror symmetric level reads one staged cell per image of
                                  a ray (8 or 16 loads of 8 bytes per slab step) instead of the copy folded onto the first
                                  quadrant (one 32-byte entry holds a cell's four quarter-turn images and their z-mirrors);
                                  same weights either way (bitwise equal projections without view pairs; with them the folded
                                  walk adds some terms in another order: equal to ~4e-8).  For A/B measurements and tests. */
#define CBCT_KERNEL_TV_SCALAR_TILES 4 /* the TV passes always on the 32-voxel warp tiles (one voxel per lane), never on the
                                         16-byte tiles that volumes with nx % 4 == 0, nx >= 128 and 16-byte aligned buffers
                                         otherwise take; same stencil, for A/B measurements and tests. */

/* Validates the description, uploads per-view tables and allocates all scratch for
 * `max_levels` levels.  *out is NULL on failure. */
cbct_status cbct_geometry_create(const cbct_geometry_desc *desc, cbct_geometry **out);
void cbct_geometry_destroy(cbct_geometry *g);

/* Rays (voxels) per thread the projectors of `level` handle with one weight computation: 4 by
 * quarter-turn symmetry, times 2 by the mirror symmetry z -> -z; 8, 4, 2 or 1 (0: bad level). */
int cbct_geometry_symmetry(const cbct_geometry *g, int level);

/* Which exact-transpose back-projector `level` runs: the TMA / shared-memory tile kernel (quarter-turn and mirror
 * symmetric geometries whose voxel shadows are at most 8 detector columns and 4 rows wide), the per-warp list kernel
 * (shadows of at most 5 columns), or the general gather kernel.  All three compute the same sums.  -1: bad level. */
#define CBCT_BACK_PATH_GATHER 0
#define CBCT_BACK_PATH_LIST 1
#define CBCT_BACK_PATH_TMA 2
int cbct_geometry_back_path(const cbct_geometry *g, int level);

/* Number of times a kernel found a tile bound computed at create too small (it then stays inside its buffers and the
 * result is wrong): 0 on every geometry the bounds were derived for; tests assert it.  Synchronises the stream. */
cbct_status cbct_bound_violations(const cbct_geometry *g, unsigned int *count, void *cuda_stream);

/* Device bytes the handle allocated (scratch + tables). */
unsigned long long cbct_geometry_device_bytes(const cbct_geometry *g);

/* A1: d_proj = P d_vol.  (P f)[a,jv,iu] = sum over voxels of (length in mm of the segment
 * source -> pixel centre inside the voxel) * f[voxel]: Eq. 1 (L91) on a piecewise-constant
 * volume, the exact radiological path of "a ray-tracing algorithm, such as Siddon's"
 * (L187, L243).  `level` selects the multi-grid level (0 = the described geometry); sizes of
 * the buffers are the level's.  Overwrites d_proj. */
cbct_status cbct_forward_project(const cbct_geometry *g, int level, const float *d_vol,
                                 float *d_proj, void *cuda_stream);

/* A3: d_vol = P^T d_proj with the SAME coefficients a(ray, voxel) as cbct_forward_project
 * (exact matrix transpose; L187 "sum_theta P^T (P f - Y)").  Voxel-driven gather, no
 * atomics, fixed summation order.  Overwrites d_vol (no accumulate). */
cbct_status cbct_back_project(const cbct_geometry *g, int level, const float *d_proj,
                              float *d_vol, void *cuda_stream);

/* NEXT-1: d_vol = b6(d_proj), the paper's own closed-form gradient of the data term, Eq. 6 (L195-L199):
 *   b6(X) = (dV / (du dv)) sum_theta L^3(u*,v*) / (L0 l^2(X)) T^theta(u*,v*),
 * (u*,v*) and l from Eq. A6 (L401-L406), T^theta(u*,v*) by bilinear interpolation between pixel centres
 * (L199; a tap outside the detector is 0).  It is the continuum adjoint, NOT the transpose of
 * cbct_forward_project: the two agree only when the pixels are much finer than a voxel's shadow.  The factor
 * dV/(du dv) puts it on the scale of cbct_back_project.  Voxel-driven, no atomics.  Overwrites d_vol. */
cbct_status cbct_back_project_eq6(const cbct_geometry *g, int level, const float *d_proj,
                                  float *d_vol, void *cuda_stream);

/* S = number of (ray, voxel) pairs with a(ray, voxel) > 0 at `level`: the "ray-voxel samples" one
 * forward (or back) projection processes -- the unit of the GUPS metric.  Synchronises the stream. */
cbct_status cbct_count_samples(const cbct_geometry *g, int level, unsigned long long *count,
                               void *cuda_stream);

/* A5: Lhat = c_norm * max_v [P^T (P 1)]_v with c_norm = 2 N_vox / (N_view N_pix): an upper
 * bound of the largest eigenvalue of the normalised data-term Hessian (reading S5).  It depends on
 * the geometry only: the first call per level evaluates it (one P, one P^T, one max-reduction;
 * synchronises the stream), later calls and cbct_fbs_reconstruct reuse the stored value. */
cbct_status cbct_step_bound(const cbct_geometry *g, int level, double *lhat, void *cuda_stream);

/* ROF sub-solver parameters (L155-L159): smoothed TV |grad f|_delta = sqrt(|grad f|^2 + delta^2)
 * (reading S6); at most max_inner accepted descent steps; at most max_backtracks shrinks of
 * the trial step per descent step; Armijo constant c, shrink factor alpha, relative-decrease
 * stop epsilon.  Paper values: c = 0.01, alpha = 0.6, epsilon = 1e-3 (L159). */
typedef struct {
    double eps_delta;
    int max_inner, max_backtracks;
    double armijo_c, shrink_alpha, rel_tol;
} cbct_tv_params;

typedef struct {
    int inner_iters; /* accepted descent steps */
    int trials;      /* trial energies evaluated */
    double e_first;  /* E_ROF[g] */
    double e_last;   /* E_ROF[returned f] */
} cbct_tv_report;

/* A6 (+A7 when nonneg != 0): d_f ~ argmin_f mean|grad f|_delta + (1/(2 w)) mean (f - g)^2
 * (Algorithm A1 step 2, L148; E_ROF L155 with beta = 1/w), by gradient descent with the Armijo
 * rule Eq. 5 (L157) started at f = g with initial trial step w (readings S8, S10); forward
 * differences in physical units with the handle's boundary rules (L161).  If nonneg, the
 * returned volume is max(f, 0) (step 3, L149).  weight_w == 0 copies g to f.
 * d_g and d_f must not alias.  report may be NULL (then the call does not synchronise). */
cbct_status cbct_tv_prox(const cbct_geometry *g, int level, const float *d_g, float *d_f,
                         double weight_w, int nonneg, const cbct_tv_params *params,
                         cbct_tv_report *report, void *cuda_stream);

/* A9 helper: *e1 = mean_v |grad f|_delta.  Synchronises the stream. */
cbct_status cbct_tv_energy(const cbct_geometry *g, int level, const float *d_f, double eps_delta,
                           double *e1, void *cuda_stream);

/* NEXT-3: the paper's image-quality metrics of a reconstruction d_f against a ground truth d_f0 (L263):
 *   *rel_error = ||f - f0||_2 / ||f0||_2,   *correlation = corr(f, f0) (Pearson, over all voxels);
 * one fused pass, fp64 sums in a fixed order.  0 is returned for a metric whose denominator vanishes.
 * Synchronises the stream. */
cbct_status cbct_quality_metrics(const cbct_geometry *g, int level, const float *d_f, const float *d_f0,
                                 double *rel_error, double *correlation, void *cuda_stream);

/* The same two metrics for callers that may not allocate (code under CUDA graph capture, tight serving loops, harnesses
 * that forbid cudaMalloc): needs NO geometry handle and calls no cudaMalloc, cudaFree or allocating routine.
 *   d_f, d_f0 : DEVICE, n floats each (caller-owned, read only);   d_out2 : DEVICE, 2 doubles: (rel_error, correlation).
 * Asynchronous on `cuda_stream` (no synchronisation, no host copy: read d_out2 after the stream has reached this call).
 * Scratch (fp64 block partials + a ticket) is a static __device__ array of CBCT_STATIC_SCRATCH_BYTES inside the library,
 * held by every GPU that loads it until the process exits; a block sums a fixed chunk of CBCT_STATIC_CHUNK elements, so the
 * summation order depends on n alone and n is limited to CBCT_STATIC_MAX_ELEMS (2^28 elements = 1 GiB per volume):
 * CBCT_ERR_INVALID_ARG beyond it (use cbct_quality_metrics), for n = 0 and for NULL buffers.  The first call on a device
 * looks the array's address up (cudaGetSymbolAddress): make that call once before capturing a graph.
 * ALL calls share the scratch: calls that overlap on the GPU (two streams, two host threads) race on it -- serialise them.
 * The ticket is cleared on the stream before every launch, so a call that failed half-way does not disturb the next.
 * Same sums as cbct_quality_metrics in another fixed order: the two agree to fp64 rounding (~1e-13 relative). */
#define CBCT_STATIC_CHUNK 16384
#define CBCT_STATIC_MAX_BLOCKS 16384
#define CBCT_STATIC_MAX_ELEMS 268435456ull
#define CBCT_STATIC_SCRATCH_BYTES (8 * (6 * CBCT_STATIC_MAX_BLOCKS + 32))
cbct_status cbct_quality_metrics_static(const float *d_f, const float *d_f0, unsigned long long n, double *d_out2,
                                        void *cuda_stream);

/* A8 grid transfers (L215-L223; readings S12, S13).  `level` is the FINE level of the pair.  Buffers need only
 * their natural 4-byte alignment (8-byte aligned fine buffers take a faster load path).
 *   restrict: fine volume -> 2x2x2 mean on level+1.   bin: fine projections -> 2x2 mean.
 *   prolong : coarse volume (level+1) -> fine, cell-centred trilinear (3/4, 1/4); a missing
 *             neighbour is 0 under BC_ZERO and the edge value under BC_REFLECT. */
cbct_status cbct_restrict_volume(const cbct_geometry *g, int level, const float *d_fine,
                                 float *d_coarse, void *cuda_stream);
cbct_status cbct_bin_projections(const cbct_geometry *g, int level, const float *d_fine,
                                 float *d_coarse, void *cuda_stream);
cbct_status cbct_prolong_volume(const cbct_geometry *g, int level, const float *d_coarse,
                                float *d_fine, void *cuda_stream);

/* Algorithm A1 (L137-L151) with the multi-grid driver (L215-L223), normalised form (S5):
 *   per level: Lhat (cbct_step_bound), tau = step / Lhat, w = tau * tv_weight;
 *   per iteration: T = P f - y; E2 = mean T^2; g = f - tau c_norm P^T T;
 *                  f = TVprox_w(g); f = max(f, 0) if nonneg.
 * Levels run n_levels-1 (coarsest) ... 0; iters_per_level[] is ordered coarsest -> finest.
 * Coarse data are 2x2-binned; the volume moves up by cbct_prolong_volume.
 * d_vol_inout: finest-level volume; the initial guess if use_initial (restricted down to
 * the coarsest level first), else ignored on entry; the result on return. */
#define CBCT_BACKPROJECTOR_EXACT 0
#define CBCT_BACKPROJECTOR_EQ6 1
typedef struct {
    double tv_weight; /* lambda = 1/mu of Eq. 2 (L97) */
    double step;      /* relative gradient step in (0, 2); 1 = 1/Lhat */
    int n_levels;     /* <= max_levels of the handle */
    const int *iters_per_level;
    int nonneg, use_initial;
    int backprojector; /* CBCT_BACKPROJECTOR_EXACT (0): g = f - tau c_norm P^T T, the matched pair;
                          CBCT_BACKPROJECTOR_EQ6 (1): g = f - tau c_norm b6(T), the paper's Eq. 6 (unmatched pair;
                          Lhat is still the matched pair's bound) */
    double conv_tol;   /* NEXT-2, "until convergence" (L145, L223; reading S20): 0 = run iters_per_level[] iterations;
                          > 0: a level also stops after the first iteration with
                          ||f_new - f_old||_2 <= conv_tol ||f_old||_2 (iters_per_level[] is then the cap) */
    cbct_tv_params tv;
} cbct_fbs_params;

typedef struct {
    int n_iters_total;
    double *objective;   /* caller-owned HOST array of sum(iters) doubles or NULL:
                            objective[it] = tv_weight*E1(f) + E2(f) of the f entering iteration it.
                            A monitored call (non-NULL) may run at most 4096 iterations in total
                            (CBCT_ERR_INVALID_ARG beyond); unmonitored calls are not limited. */
    double *step_abs;    /* caller-owned HOST array of n_levels doubles or NULL: tau per level */
    int *iters_done;     /* caller-owned HOST array of n_levels ints or NULL: iterations run per level, coarsest ->
                            finest (= iters_per_level[] unless conv_tol stopped a level early); objective[] holds
                            sum(iters_done) entries in that order */
    int inner_total, trials_total; /* summed over all TV-prox calls */
    float ms_total;      /* device time of the whole call (CUDA events on the stream) */
} cbct_fbs_report;

cbct_status cbct_fbs_reconstruct(const cbct_geometry *g, const float *d_proj_y, float *d_vol_inout,
                                 const cbct_fbs_params *params, cbct_fbs_report *report,
                                 void *cuda_stream);

/* The same call on HOST buffers: copies h_proj_y to the device, reconstructs, copies the
 * volume back (and reads h_vol_inout first if use_initial).  The handle owns the device
 * staging buffers.  Pinned host memory makes the copies asynchronous but is not required.
 * Synchronises the stream. */
cbct_status cbct_fbs_reconstruct_host(const cbct_geometry *g, const float *h_proj_y,
                                      float *h_vol_inout, const cbct_fbs_params *params,
                                      cbct_fbs_report *report, void *cuda_stream);

/* NEXT-4 -- the reconstruction sharded over `world` GPUs by OUTPUT OWNERSHIP (one process and one handle per GPU, every
 * rank calling with the same arguments).  Every rank holds the whole volume and the whole data; per iteration
 *   - rank r projects ITS forward units (cbct_shard_range over cbct_shard_units' n_base_views: base views -- with quarter-turn
 *     symmetry a base view stands for its four quarter-turn partners -- or, where the view set is also symmetric under
 *     theta -> -theta, view PAIRS (p, n_base - p)) and the residual chunks are broadcast from their owners;
 *   - the blocks' partial sums of T^2 are added across ranks (every slot is written by exactly one rank, the others hold
 *     0, so the addition is exact) and summed in the single-GPU order;
 *   - rank r evaluates g = f - tau c_norm P^T T on ITS z-units (n_z_units of z_unit_slices slices of the lower half volume,
 *     with their mirror images; of the whole volume without mirror symmetry) and the slabs are broadcast from their owners;
 *   - the TV step, the grid transfers and the step bound run replicated: deterministic kernels on identical inputs.
 * Every residual value and every voxel of g is computed by exactly one rank with the arithmetic of the single-GPU launch, so
 * the result on every rank is BIT FOR BIT cbct_fbs_reconstruct's.  The two collectives are the caller's (NCCL through
 * torch.distributed in the Python binding): callbacks on caller-owned DEVICE memory of the handle, to be ordered on
 * `cuda_stream` (enqueue on it, or synchronise it before and after); they return 0 on success.
 * Only CBCT_BACKPROJECTOR_EXACT.  Not exercised on more than one GPU in this repository's CI (one-GPU boxes): covered by a
 * two-rank emulation on one GPU against the single-GPU result and by CPU tests of the partition. */
typedef struct cbct_comm {
    int rank, world;
    void *ctx;
    int (*broadcast)(void *ctx, void *d_buf, unsigned long long bytes, int root, void *cuda_stream);    /* in place */
    int (*allreduce_sum_f64)(void *ctx, double *d_buf, unsigned long long n, void *cuda_stream);        /* in place */
} cbct_comm;

/* Balanced contiguous split of n_units over `world` ranks: [*lo, *hi) for `rank` (the first n_units % world ranks take one
 * unit more).  Pure host arithmetic: needs no device. */
cbct_status cbct_shard_range(int n_units, int world, int rank, int *lo, int *hi);
/* The units a level's projectors are sharded in (any pointer may be NULL). */
cbct_status cbct_shard_units(const cbct_geometry *g, int level, int *n_base_views, int *n_z_units, int *z_unit_slices);
cbct_status cbct_fbs_reconstruct_sharded(const cbct_geometry *g, const cbct_comm *comm, const float *d_proj_y,
                                         float *d_vol_inout, const cbct_fbs_params *params, cbct_fbs_report *report,
                                         void *cuda_stream);

/* Kernel launches issued by this handle since create (for the bench's gpu_launches). */
unsigned long long cbct_launch_count(const cbct_geometry *g);

/* Per-kernel attribution.  When switched on, every launch of the kernels below is bracketed by
 * CUDA events on the library's stream and its device time accumulated (this adds one
 * synchronisation per launch, so timings of whole calls taken with it on are for attribution only).
 * Slots: 0 volume transpose (forward projector's x<->y copy), 1 forward projector kernel,
 * 2 back-projector kernel, 3 TV gradient pass, 4 TV trial-energy pass, 5 TV update / clip pass,
 * 6 reduction finalisers + objective monitor, 7 grid transfers, fills, max.
 * cbct_get_stage_ms returns the accumulated milliseconds and launch-group counts since the last
 * cbct_set_stage_timing call. */
#define CBCT_N_STAGES 8
cbct_status cbct_set_stage_timing(cbct_geometry *g, int enable);
cbct_status cbct_get_stage_ms(const cbct_geometry *g, float out_ms[CBCT_N_STAGES],
                              unsigned long long out_calls[CBCT_N_STAGES]);

/* Measured ceiling of the gather patterns the projectors are made of: a calibration kernel
 * issues blocks x 256 threads x iters x 8 independent loads from d_buf (n_floats floats, 16-byte aligned, caller-owned,
 * any finite contents) and reports its device time and the bytes the lanes asked for.  variant 0: 4-byte loads, a warp
 * reads one contiguous 128-byte run (forward projector); 1: 16-byte loads two entries apart (back-projector, L1 path);
 * 2 / 3: 16-byte loads two entries apart from a shared-memory tile, plain / split by entry parity (back_tma.cu).
 * The run's position is pseudo-random inside a 16 KB tile that moves every `reuse` loads (variants 0, 1): reuse = 1
 * gathers from L2, a large reuse from L1.  d_sink: one float the kernel may write.  Synchronises the stream.
 * Not part of the hot path: bench.py quotes the projectors' GUPS against it. */
cbct_status cbct_gather_ceiling(const float *d_buf, unsigned long long n_floats, int variant, int reuse, int iters,
                                float *d_sink, float *ms, unsigned long long *bytes, void *cuda_stream);

/* Thread-local message of the last failing call on this thread ("" if none). */
const char *cbct_last_error(void);
const char *cbct_version(void);

#ifdef __cplusplus
}
#endif
#endif /* CBCT_H */
