// geometry.cu -- handle life cycle: validation, per-level ray tables, scratch.
// A0 of the scope table: per view S, e_n, e_u, e_v.
#include <math.h>
#include <stdarg.h>
#include <stdio.h>
#include <string.h>
#include <new>
#include "cbct_internal.cuh"

static thread_local char tls_error[512] = "";

cbct_status cbct_fail(cbct_status st, const char *fmt, ...)
{
    va_list ap;
    va_start(ap, fmt);
    vsnprintf(tls_error, sizeof(tls_error), fmt, ap);
    va_end(ap);
    return st;
}

extern "C" const char *cbct_last_error(void) { return tls_error; }
extern "C" const char *cbct_version(void) { return "libcbct 0.1 (sm_100a)"; }

template <typename T>
static cbct_status dev_alloc(cbct_geometry *g, T **p, size_t n)
{
    *p = nullptr;
    if (n == 0) return CBCT_OK;
    cudaError_t e = cudaMalloc((void **)p, n * sizeof(T));
    if (e != cudaSuccess) {
        cudaGetLastError();
        return cbct_fail(CBCT_ERR_OOM, "cudaMalloc(%zu bytes): %s", n * sizeof(T), cudaGetErrorString(e));
    }
    g->device_bytes += n * sizeof(T);
    return CBCT_OK;
}

// Build the (view, iu) ray table of one level in fp64, round once to fp32.
static cbct_status build_tables(const cbct_geometry *g, Level &L, std::vector<RayU> &rays,
                                std::vector<ViewC> &views)
{
    const cbct_geometry_desc &d = g->desc;
    const LevelParams &p = L.p;
    rays.resize((size_t)p.np * p.nu);
    views.resize(p.np);
    // index coordinate of a point x (mm) on axis a:  (x - off_a)/h_a + n_a/2.0 - (n_a/2)
    const double shx = 0.5 * p.nx - p.cx, shy = 0.5 * p.ny - p.cy, shz = 0.5 * p.nz - p.cz;
    const double vmax = fmax(fabs(-0.5 * (p.nv - 1) * L.dv + d.det_off_v),
                             fabs(0.5 * (p.nv - 1) * L.dv + d.det_off_v));
    for (int a = 0; a < p.np; ++a) {
        const double t = g->angles[a], c = cos(t), s = sin(t);
        const double sxi = (-d.sad * c - d.vol_off[0]) / L.hx + shx;
        const double syi = (-d.sad * s - d.vol_off[1]) / L.hy + shy;
        ViewC vc;
        vc.c = (float)c; vc.s = (float)s;
        // half extents of a voxel along e_n and e_u, inflated so that the first-order bounds of
        // back.cu on the voxel's shadow are conservative
        vc.dn = (float)(1.01 * 0.5 * (fabs(c) * L.hx + fabs(s) * L.hy));
        vc.du = (float)(1.003 * 0.5 * (fabs(s) * L.hx + fabs(c) * L.hy));
        views[a] = vc;
        for (int iu = 0; iu < p.nu; ++iu) {
            const double u = (iu - 0.5 * (p.nu - 1)) * L.du + d.det_off_u;
            const double dxi = (d.sdd * c + u * s) / L.hx, dyi = (d.sdd * s - u * c) / L.hy;
            RayU r;
            double m, a0, sd, dd;
            if (fabs(dxi) >= fabs(dyi)) { r.drive = 0; dd = dxi; m = dyi / dxi; a0 = syi - sxi * m; sd = sxi; }
            else                        { r.drive = 1; dd = dyi; m = dxi / dyi; a0 = sxi - syi * m; sd = syi; }
            const double q = (1.0 / L.hz) / dd;
            if (fabs(vmax * q) > 1.0)
                return cbct_fail(CBCT_ERR_GEOMETRY,
                                 "view %d: a ray crosses more than one z-plane per in-plane slab "
                                 "(|v|max * hd/(hz*Dd) = %.3f > 1); voxels too flat in z for this cone angle",
                                 a, fabs(vmax * q));
            r.a0 = (float)a0; r.m = (float)m;
            r.inv_m = (r.m == 0.0f) ? 1.0e30f : (float)(1.0 / m);
            r.q = (float)q; r.sd = (float)sd; r.inv_dd = (float)(1.0 / fabs(dd));
            r.c_l = (float)(d.sdd * d.sdd + u * u);
            rays[(size_t)a * p.nu + iu] = r;
        }
    }
    (void)shz;
    return CBCT_OK;
}

static cbct_status validate(const cbct_geometry_desc *d)
{
    if (d->nx <= 0 || d->ny <= 0 || d->nz <= 0 || d->nu <= 0 || d->nv <= 0 || d->n_proj <= 0)
        return cbct_fail(CBCT_ERR_INVALID_ARG, "non-positive dimension");
    if (!(d->hx > 0 && d->hy > 0 && d->hz > 0 && d->du > 0 && d->dv > 0))
        return cbct_fail(CBCT_ERR_INVALID_ARG, "non-positive voxel size or pixel pitch");
    if (d->max_levels < 1 || d->max_levels > 8)
        return cbct_fail(CBCT_ERR_INVALID_ARG, "max_levels must be in 1..8");
    int div = 1 << (d->max_levels - 1);
    if (d->nx % div || d->ny % div || d->nz % div || d->nu % div || d->nv % div)
        return cbct_fail(CBCT_ERR_INVALID_ARG, "every volume and detector dimension must be divisible by 2^(max_levels-1) = %d", div);
    if ((d->bc_xy != CBCT_BC_ZERO && d->bc_xy != CBCT_BC_REFLECT) ||
        (d->bc_z != CBCT_BC_ZERO && d->bc_z != CBCT_BC_REFLECT))
        return cbct_fail(CBCT_ERR_INVALID_ARG, "boundary condition must be CBCT_BC_ZERO or CBCT_BC_REFLECT");
    if (!(d->sad > 0 && d->sdd > d->sad))
        return cbct_fail(CBCT_ERR_GEOMETRY, "need 0 < sad < sdd");
    if ((long long)d->nx * d->ny * d->nz >= (1LL << 31) || (long long)d->nu * d->nv * d->n_proj >= (1LL << 31))
        return cbct_fail(CBCT_ERR_INVALID_ARG, "volume or projection stack has 2^31 or more elements");
    // the volume must stay strictly between the source and the detector plane
    double rx = 0.5 * d->nx * d->hx + fabs(d->vol_off[0]), ry = 0.5 * d->ny * d->hy + fabs(d->vol_off[1]);
    double r = sqrt(rx * rx + ry * ry);
    if (r >= d->sad || r >= d->sdd - d->sad)
        return cbct_fail(CBCT_ERR_GEOMETRY, "volume (in-plane radius %.1f mm) reaches the source orbit (%.1f) or the detector plane (%.1f)",
                         r, d->sad, d->sdd - d->sad);
    return CBCT_OK;
}

static void free_all(cbct_geometry *g)
{
    if (!g) return;
    for (Level &L : g->levels) {
        cudaFree(L.d_rayu); cudaFree(L.d_view); cudaFree(L.d_cs); cudaFree(L.d_stage); cudaFree(L.d_T); cudaFree(L.bt.d_lists); cudaFree(L.bt.d_hdrs);
        cudaFree(L.d_g); cudaFree(L.d_d); cudaFree(L.d_f2); cudaFree(L.d_f); cudaFree(L.d_prev); cudaFree(L.d_y);
    }
    cudaFree(g->d_partials); cudaFree(g->d_scalars); cudaFree(g->d_objective); cudaFree(g->d_counter); cudaFree(g->d_errflag);
    if (g->h_scalars) cudaFreeHost(g->h_scalars);
    for (int i = 0; i < 5; ++i) if (g->ev[i]) cudaEventDestroy(g->ev[i]);
    delete g;
}

extern "C" void cbct_geometry_destroy(cbct_geometry *g) { free_all(g); }

extern "C" cbct_status cbct_geometry_create(const cbct_geometry_desc *desc, cbct_geometry **out)
{
    if (out) *out = nullptr;
    if (!desc || !out) return cbct_fail(CBCT_ERR_INVALID_ARG, "NULL argument");
    cbct_status st = validate(desc);
    if (st != CBCT_OK) return st;

    int dev = 0, n_dev = 0;
    if (cudaGetDeviceCount(&n_dev) != cudaSuccess || n_dev == 0) {
        cudaGetLastError();
        return cbct_fail(CBCT_ERR_UNSUPPORTED, "no CUDA device: libcbct has no CPU fallback");
    }
    CBCT_CUDA(cudaGetDevice(&dev));
    cudaDeviceProp prop;
    CBCT_CUDA(cudaGetDeviceProperties(&prop, dev));
    if (prop.major != 10)
        return cbct_fail(CBCT_ERR_UNSUPPORTED, "device '%s' is sm_%d%d; libcbct is built for sm_100a only",
                         prop.name, prop.major, prop.minor);

    cbct_geometry *g = new (std::nothrow) cbct_geometry();
    if (!g) return cbct_fail(CBCT_ERR_OOM, "host allocation failed");
    g->desc = *desc;
    g->allow_symmetry = desc->no_symmetry ? 0 : 1;
    g->disable_tma = (desc->kernel_flags & CBCT_KERNEL_NO_TMA) ? 1 : 0;
    g->host_armijo = (desc->kernel_flags & CBCT_KERNEL_HOST_ARMIJO) ? 1 : 0;
    g->tv_scalar_tiles = (desc->kernel_flags & CBCT_KERNEL_TV_SCALAR_TILES) ? 1 : 0;
    g->back_lists_on_the_fly = (desc->kernel_flags & CBCT_KERNEL_BACK_LISTS_ON_THE_FLY) ? 1 : 0;
    g->no_reflection = (desc->kernel_flags & CBCT_KERNEL_NO_REFLECTION) ? 1 : 0;
    g->no_fold = (desc->kernel_flags & CBCT_KERNEL_NO_FOLD) ? 1 : 0;
    {   // the cooperative TV-prox kernel needs cooperative launches (every sm_100 device has them; checked all the same)
        int coop = 0;
        if (cudaDeviceGetAttribute(&coop, cudaDevAttrCooperativeLaunch, dev) != cudaSuccess || !coop) g->host_armijo = 1;
    }
    g->sm_count = prop.multiProcessorCount;
    g->angles.resize(desc->n_proj);
    for (int a = 0; a < desc->n_proj; ++a)
        g->angles[a] = desc->angles_rad ? desc->angles_rad[a] : 2.0 * M_PI * a / desc->n_proj;
    g->desc.angles_rad = nullptr;

    st = dev_alloc(g, &g->d_errflag, (size_t)1);
    if (st != CBCT_OK) { free_all(g); return st; }
    // zeroed before the levels are planned: the tables bt_plan_level builds count violated tile bounds in it
    if (cudaMemset(g->d_errflag, 0, sizeof(unsigned int)) != cudaSuccess) { free_all(g); return cbct_fail(CBCT_ERR_CUDA, "memset failed"); }
    g->levels.resize(desc->max_levels);
    for (int l = 0; l < desc->max_levels; ++l) {
        Level &L = g->levels[l];
        const int f = 1 << l;
        LevelParams &p = L.p;
        p.nx = desc->nx / f; p.ny = desc->ny / f; p.nz = desc->nz / f;
        p.nu = desc->nu / f; p.nv = desc->nv / f; p.np = desc->n_proj;
        p.cx = p.nx / 2; p.cy = p.ny / 2; p.cz = p.nz / 2;
        L.hx = desc->hx * f; L.hy = desc->hy * f; L.hz = desc->hz * f;
        L.du = desc->du * f; L.dv = desc->dv * f;
        p.hx = (float)L.hx; p.hy = (float)L.hy; p.hz = (float)L.hz;
        p.x0 = (float)(-0.5 * (p.nx - 1) * L.hx + desc->vol_off[0]);
        p.y0 = (float)(-0.5 * (p.ny - 1) * L.hy + desc->vol_off[1]);
        p.z0 = (float)(-0.5 * (p.nz - 1) * L.hz + desc->vol_off[2]);
        p.u0 = (float)(-0.5 * (p.nu - 1) * L.du + desc->det_off_u);
        p.v0 = (float)(-0.5 * (p.nv - 1) * L.dv + desc->det_off_v);
        p.du = (float)L.du; p.dv = (float)L.dv;
        p.inv_du = (float)(1.0 / L.du); p.inv_dv = (float)(1.0 / L.dv);
        p.sz = (float)((0.0 - desc->vol_off[2]) / L.hz + (0.5 * p.nz - p.cz));
        p.sad = (float)desc->sad; p.sdd = (float)desc->sdd;
        p.bc_xy = desc->bc_xy; p.bc_z = desc->bc_z;
        L.nvox = (size_t)p.nx * p.ny * p.nz;
        L.nray = (size_t)p.nu * p.nv * p.np;
        // quarter-turn symmetry: square centred in-plane grid, views a and a + np/4 a quarter turn apart
        p.nsym = 1;
        if (g->allow_symmetry && p.nx == p.ny && p.nx % 2 == 0 && L.hx == L.hy && desc->vol_off[0] == 0.0 &&
            desc->vol_off[1] == 0.0 && p.np % 4 == 0) {
            bool ok = true;
            const int nb = p.np / 4;
            for (int a = 0; a + nb < p.np && ok; ++a)
                ok = fabs(g->angles[a + nb] - g->angles[a] - 0.5 * M_PI) < 1e-12;
            if (ok) p.nsym = 4;
        }
        p.nbase = p.np / p.nsym;
        // reflection symmetry theta -> -theta on top of the quarter turns: theta_0 = 0 and theta_a + theta_(nbase-a) = 90 degrees,
        // detector centred in u with an even column count (column iu <-> nu-1-iu)
        p.nrefl = 1; p.npairs = p.nbase;
        if (p.nsym == 4 && !g->no_reflection && desc->det_off_u == 0.0 && p.nu % 2 == 0 && fabs(g->angles[0]) < 1e-12) {
            bool ok = true;
            for (int a = 1; a < p.nbase && ok; ++a)
                ok = fabs(g->angles[a] + g->angles[p.nbase - a] - 0.5 * M_PI) < 1e-12;
            if (ok) { p.nrefl = 2; p.npairs = p.nbase / 2 + 1; }
        }
        // mirror symmetry z -> -z: volume centred in z, detector centred in v, even sizes
        p.nmir = (g->allow_symmetry && desc->vol_off[2] == 0.0 && desc->det_off_v == 0.0 && p.nz % 2 == 0 && p.nv % 2 == 0) ? 2 : 1;

        // staged copy [nx+2PM][ny+2PM][nzP], z fastest: floats with nzP = nz + 2PZ, or (mirror symmetry) float2
        // pairs (f(k), f(nz-1-k)) with nzP = nz/2 + 2PZ; strides in cells
        p.nyP = p.ny + 2 * PAD_M;
        p.nzP = (p.nmir == 2 ? p.nz / 2 : p.nz) + 2 * PAD_Z;
        p.jstride = p.nzP; p.istride = p.nyP * p.nzP;
        L.stage_elems = (size_t)(p.nx + 2 * PAD_M) * p.nyP * p.nzP * p.nmir;
        p.stage_cells = (int)(L.stage_elems / p.nmir);
        // quarter-turn + mirror symmetric levels: the copy folded onto the first quadrant, 8 floats per canonical cell (forward.cu)
        p.fold = (p.nsym == 4 && p.nmir == 2 && !g->no_fold) ? 1 : 0;
        p.nhP = p.nx / 2 + PAD_M; p.fjs = p.nzP; p.fis = p.nhP * p.nzP;
        if (p.fold) {
            L.stage_elems = (size_t)p.nhP * p.nhP * p.nzP * 8;
            p.stage_cells = (int)(L.stage_elems / 8);
        }
        p.t_entries = (int)(L.nray / p.nsym);
        p.tP = 1; p.tXP = p.nv;
        if (L.stage_elems >= (size_t)1 << 31) { free_all(g); return cbct_fail(CBCT_ERR_INVALID_ARG, "padded volume copy exceeds 2^31 elements"); }

        std::vector<RayU> rays;
        std::vector<ViewC> views;
        st = build_tables(g, L, rays, views);
        if (st != CBCT_OK) { free_all(g); return st; }
#define TRY(x) do { st = (x); if (st != CBCT_OK) { free_all(g); return st; } } while (0)
        {   // widest shadow of a voxel square on the detector's u axis, in columns: back.cu's W at the largest
            // magnification (volume corner nearest to the source) and fan angle, as that kernel inflates it
            double rx = 0.5 * p.nx * L.hx + fabs(desc->vol_off[0]), ry = 0.5 * p.ny * L.hy + fabs(desc->vol_off[1]);
            double rmax = sqrt(rx * rx + ry * ry), mag = desc->sdd / (desc->sad - rmax);
            double umax = 0.5 * p.nu * L.du + fabs(desc->det_off_u), tn = fmax(umax / desc->sdd, rmax / (desc->sad - rmax));
            double dn = 0, du = 0;
            for (const ViewC &v : views) { dn = fmax(dn, v.dn); du = fmax(du, v.du); }
            double W = mag * (tn * dn + du);
            L.back_maxc = (int)floor(2.0 * W / L.du + 0.04) + 1;       // integers in an interval of that length
        }
        TRY(dev_alloc(g, &L.d_rayu, rays.size()));
        TRY(dev_alloc(g, &L.d_view, views.size()));
        TRY(dev_alloc(g, &L.d_cs, views.size()));
        TRY(dev_alloc(g, &L.d_stage, L.stage_elems));
        if (cudaMemset(L.d_stage, 0, L.stage_elems * sizeof(float)) != cudaSuccess) { free_all(g); return cbct_fail(CBCT_ERR_CUDA, "memset of the staged volume failed"); }
        TRY(dev_alloc(g, &L.d_T, L.nray));
        TRY(dev_alloc(g, &L.d_g, L.nvox));
        TRY(dev_alloc(g, &L.d_d, L.nvox));
        TRY(dev_alloc(g, &L.d_f2, L.nvox));
        TRY(dev_alloc(g, &L.d_f, L.nvox));
        TRY(dev_alloc(g, &L.d_prev, L.nvox));
        TRY(dev_alloc(g, &L.d_y, L.nray));
        cudaError_t e = cudaMemcpy(L.d_rayu, rays.data(), rays.size() * sizeof(RayU), cudaMemcpyHostToDevice);
        if (e == cudaSuccess)
            e = cudaMemcpy(L.d_view, views.data(), views.size() * sizeof(ViewC), cudaMemcpyHostToDevice);
        if (e == cudaSuccess) {
            std::vector<double2> cs(p.np);
            for (int a = 0; a < p.np; ++a) cs[a] = make_double2(cos(g->angles[a]), sin(g->angles[a]));
            e = cudaMemcpy(L.d_cs, cs.data(), cs.size() * sizeof(double2), cudaMemcpyHostToDevice);
        }
        if (e != cudaSuccess) { free_all(g); return cbct_fail(CBCT_ERR_CUDA, "table upload: %s", cudaGetErrorString(e)); }
        TRY(bt_plan_level(g, L));       // the TMA back-projector's tiles and the residual stack's layout (back_tma.cu)
    }
    {
        size_t need = 1024;
        for (const Level &L : g->levels) {
            const LevelParams &p = L.p;
            size_t fwd = (size_t)((p.nu + 31) / 32) * ((p.nv + 7) / 8) * p.np;     // count_samples_kernel blocks
            size_t fw2 = (size_t)((p.nu + 7) / 8) * ((p.nv + 31) / 32) * p.np;     // forward_kernel blocks (upper bound)
            if (fw2 > fwd) fwd = fw2;
            size_t tv = (size_t)((p.nx + 31) / 32) * ((p.ny + 15) / 16) * ((p.nz + 3) / 4);   // tv.cu blocks, shortest march
            if (fwd > need) need = fwd;
            if (tv > need) need = tv;
        }
        g->partials_stride = (int)need;
    }
    TRY(dev_alloc(g, &g->d_partials, (size_t)8 * g->partials_stride));
    TRY(dev_alloc(g, &g->d_scalars, (size_t)kScalars));
    TRY(dev_alloc(g, &g->d_counter, (size_t)4));        // [0] ticket of the fused reductions, [1..2] tile tickets of the cooperative TV-prox
    if (cudaMemset(g->d_counter, 0, 4 * sizeof(unsigned int)) != cudaSuccess || cudaMemset(g->d_scalars, 0, sizeof(double) * kScalars) != cudaSuccess) { free_all(g); return cbct_fail(CBCT_ERR_CUDA, "memset of the reduction scalars failed"); }
    g->objective_cap = 4096;
    TRY(dev_alloc(g, &g->d_objective, (size_t)2 * g->objective_cap));
#undef TRY
    if (cudaMallocHost((void **)&g->h_scalars, sizeof(double) * kScalars) != cudaSuccess) {
        free_all(g);
        return cbct_fail(CBCT_ERR_OOM, "pinned host allocation failed");
    }
    for (int i = 0; i < 5; ++i)
        if (cudaEventCreate(&g->ev[i]) != cudaSuccess) { free_all(g); return cbct_fail(CBCT_ERR_CUDA, "event create failed"); }
    tls_error[0] = 0;
    *out = g;
    return CBCT_OK;
}

extern "C" int cbct_geometry_symmetry(const cbct_geometry *g, int level)
{
    const Level *L = get_level(g, level);
    return L ? L->p.nsym * L->p.nmir : 0;
}

extern "C" int cbct_geometry_back_path(const cbct_geometry *g, int level)
{
    const Level *L = get_level(g, level);
    if (!L) return -1;
    if (L->bt.ok) return CBCT_BACK_PATH_TMA;
    return L->back_maxc <= 5 ? CBCT_BACK_PATH_LIST : CBCT_BACK_PATH_GATHER;
}

extern "C" cbct_status cbct_bound_violations(const cbct_geometry *g, unsigned int *count, void *cuda_stream)
{
    if (!g || !count) return cbct_fail(CBCT_ERR_INVALID_ARG, "cbct_bound_violations: NULL argument");
    cudaStream_t st = (cudaStream_t)cuda_stream;
    CBCT_CUDA(cudaMemcpyAsync(count, g->d_errflag, sizeof(unsigned int), cudaMemcpyDeviceToHost, st));
    CBCT_CUDA(cudaStreamSynchronize(st));
    return CBCT_OK;
}

extern "C" unsigned long long cbct_geometry_device_bytes(const cbct_geometry *g) { return g ? g->device_bytes : 0ULL; }
extern "C" unsigned long long cbct_launch_count(const cbct_geometry *g) { return g ? g->launches : 0ULL; }

extern "C" cbct_status cbct_set_stage_timing(cbct_geometry *g, int enable)
{
    if (!g) return cbct_fail(CBCT_ERR_INVALID_ARG, "NULL handle");
    g->stage_timing = enable ? 1 : 0;
    for (int i = 0; i < CBCT_N_STAGES; ++i) { g->stage_ms[i] = 0.f; g->stage_calls[i] = 0; }
    return CBCT_OK;
}

extern "C" cbct_status cbct_get_stage_ms(const cbct_geometry *g, float out_ms[CBCT_N_STAGES],
                                         unsigned long long out_calls[CBCT_N_STAGES])
{
    if (!g || !out_ms) return cbct_fail(CBCT_ERR_INVALID_ARG, "NULL argument");
    for (int i = 0; i < CBCT_N_STAGES; ++i) {
        out_ms[i] = g->stage_ms[i];
        if (out_calls) out_calls[i] = g->stage_calls[i];
    }
    return CBCT_OK;
}
