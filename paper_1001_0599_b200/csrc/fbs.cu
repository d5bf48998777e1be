// fbs.cu -- A4/A5/A9 and the drivers: Algorithm A1 inside the
// coarse-to-fine multi-grid loop (L215-L223), in the normalised discrete form of DESIGN.md
// reading S5:
//   E2 = mean_{view,pixel} (P f - y)^2,  c_norm = 2 N_vox / (N_view N_pix),
//   step 1 (L147): g = f - tau c_norm P^T (P f - y)
//   step 2 (L148): f = TVprox_w(g),  w = tau * tv_weight
//   step 3 (L149): f = max(f, 0)
//   tau = step / Lhat,  Lhat = c_norm max_v [P^T (P 1)]_v   (row-sum bound, once per level)
// Every stage is a kernel of this library; the host only sequences launches.
#include <math.h>
#include "cbct_internal.cuh"
#include "reduce.cuh"

namespace {

// The forward projection of the NEXT iteration, queued behind the first TV trial pass of this one (run_tv_prox, TvAhead):
// the trial leaves the candidate result in f, and in the usual case -- first step accepted and last -- that is the result,
// so the device goes straight on while the host is still reading the trial's sums.  Otherwise the projection is redone.
struct ForwardAhead {
    const cbct_geometry *g;
    const Level *L;
    const float *f, *y;
    int mode;
    double *sum_slot;
    cudaStream_t st;
};
cbct_status forward_ahead(void *ctx)
{
    const ForwardAhead *a = static_cast<const ForwardAhead *>(ctx);
    return launch_forward(a->g, *a->L, a->f, a->y, a->L->d_T, a->mode, a->sum_slot, a->st);
}

// Lhat of one level (cached in the handle after the first evaluation: it depends on the geometry only).
cbct_status step_bound_level(const cbct_geometry *g, const Level &L, double *lhat, cudaStream_t st)
{
    cbct_status s;
    if (L.lhat > 0.0) { *lhat = L.lhat; return CBCT_OK; }
    if ((s = launch_fill(g, L.d_g, L.nvox, 1.0f, st)) != CBCT_OK) return s;
    if ((s = launch_forward(g, L, L.d_g, nullptr, L.d_T, 2, nullptr, st)) != CBCT_OK) return s;   // L * (P 1)
    if ((s = launch_back(g, L, L.d_T, 1, nullptr, 0.0f, L.d_d, st)) != CBCT_OK) return s;
    if ((s = launch_max(g, L.d_d, L.nvox, g->d_scalars + 9, st)) != CBCT_OK) return s;
    CBCT_CUDA(cudaMemcpyAsync(g->h_scalars + 9, g->d_scalars + 9, sizeof(double), cudaMemcpyDeviceToHost, st));
    CBCT_CUDA(cudaStreamSynchronize(st));
    const double c_norm = 2.0 * (double)L.nvox / (double)L.nray;
    *lhat = c_norm * g->h_scalars[9];
    if (*lhat > 0.0) L.lhat = *lhat;
    return CBCT_OK;
}

cbct_status check_params(const cbct_geometry *g, const cbct_fbs_params *p)
{
    if (!g || !p) return cbct_fail(CBCT_ERR_INVALID_ARG, "cbct_fbs_reconstruct: NULL handle or params");
    if (p->n_levels < 1 || p->n_levels > (int)g->levels.size())
        return cbct_fail(CBCT_ERR_INVALID_ARG, "cbct_fbs_reconstruct: n_levels = %d but the handle provisions %d",
                         p->n_levels, (int)g->levels.size());
    if (!p->iters_per_level) return cbct_fail(CBCT_ERR_INVALID_ARG, "cbct_fbs_reconstruct: iters_per_level is NULL");
    long total = 0;
    for (int l = 0; l < p->n_levels; ++l) {
        if (p->iters_per_level[l] < 0) return cbct_fail(CBCT_ERR_INVALID_ARG, "cbct_fbs_reconstruct: negative iteration count");
        total += p->iters_per_level[l];
    }
    (void)total;
    if (!(p->tv_weight >= 0.0) || !(p->step > 0.0 && p->step < 2.0))
        return cbct_fail(CBCT_ERR_INVALID_ARG, "cbct_fbs_reconstruct: need tv_weight >= 0 and 0 < step < 2");
    if (!(p->conv_tol >= 0.0)) return cbct_fail(CBCT_ERR_INVALID_ARG, "cbct_fbs_reconstruct: conv_tol must be >= 0");
    if (p->backprojector != CBCT_BACKPROJECTOR_EXACT && p->backprojector != CBCT_BACKPROJECTOR_EQ6)
        return cbct_fail(CBCT_ERR_INVALID_ARG, "cbct_fbs_reconstruct: unknown backprojector %d", p->backprojector);
    if (p->tv.max_inner < 0 || p->tv.max_backtracks < 0 || !(p->tv.shrink_alpha > 0.0 && p->tv.shrink_alpha < 1.0))
        return cbct_fail(CBCT_ERR_INVALID_ARG, "cbct_fbs_reconstruct: bad TV parameters");
    return CBCT_OK;
}

// ---- NEXT-4: the two projectors sharded by output ownership ------------------------------------
// Every rank holds the whole volume and the whole data.  A rank computes the residual of ITS base views (with their
// quarter-turn partners) and g = f - tau c_norm P^T T on ITS z-units (with their mirror images); the residual chunks and
// the slabs of g are then broadcast from their owners, and the blocks' partial sums of T^2 are added across ranks (each
// slot is written by one rank, the others hold 0: exact) and summed in the single-GPU order.  Every element is computed
// by exactly one rank with the arithmetic of the single-GPU launch, so the volume is bit for bit the single-GPU one; the TV
// step, the transfers and the step bound run replicated (deterministic: every rank gets the same bits).
void shard_range(int n, int world, int rank, int *lo, int *hi)
{
    const int q = n / world, r = n % world;             // the first r ranks take one unit more
    *lo = rank * q + (rank < r ? rank : r);
    *hi = *lo + q + (rank < r ? 1 : 0);
}

#define CBCT_COMM(expr)                                                                                  \
    do {                                                                                                 \
        if ((expr) != 0) return cbct_fail(CBCT_ERR_CUDA, "communicator callback failed: %s", #expr);     \
    } while (0)

// T = L inv_dd (P f - y) on every rank, and sum T^2 / (L inv_dd)^2 in *d_sum_sq
cbct_status sharded_forward(const cbct_geometry *g, const Level &L, const cbct_comm *cm, const float *f, const float *y,
                            double *d_sum_sq, cudaStream_t st)
{
    const LevelParams &P = L.p;
    cbct_status s;
    Shard sh = {0, 0, 0, 0};
    const int units = forward_units(L);         // base views, or view pairs (p, n_base - p) where the walk serves the reflections too
    shard_range(units, cm->world, cm->rank, &sh.base_lo, &sh.base_hi);
    const size_t nblk = (size_t)((P.nu + 7) / 8) * units * ((P.nv / P.nmir + 31) / 32);         // forward.cu's full grid
    if (nblk > (size_t)g->partials_stride) return cbct_fail(CBCT_ERR_INVALID_ARG, "projection stack too large for the reduction buffer");
    CBCT_CUDA(cudaMemsetAsync(g->d_partials, 0, nblk * sizeof(double), st));
    if ((s = launch_forward(g, L, f, y, L.d_T, 1, nullptr, st, &sh)) != CBCT_OK) return s;
    const size_t per_base = (size_t)P.nu * P.nv * P.nsym * sizeof(float);                       // one base view of the stack
    for (int r = 0; r < cm->world; ++r) {
        int lo, hi;
        shard_range(units, cm->world, r, &lo, &hi);
        if (hi <= lo) continue;
        if (units == P.nbase) {
            CBCT_COMM(cm->broadcast(cm->ctx, (char *)L.d_T + (size_t)lo * per_base, (unsigned long long)(hi - lo) * per_base, r, st));
        } else {
            // pairs lo .. hi-1 own the base views lo .. hi-1 and their partners n_base-(hi-1) .. n_base-lo (pair 0 and the
            // middle pair of an even n_base are their own partners): two contiguous runs, trimmed where they meet or repeat
            const int a_hi = hi < P.nbase ? hi : P.nbase;                                        // first run: [lo, a_hi)
            CBCT_COMM(cm->broadcast(cm->ctx, (char *)L.d_T + (size_t)lo * per_base, (unsigned long long)(a_hi - lo) * per_base, r, st));
            int p_lo = P.nbase - (hi - 1), p_hi = P.nbase - lo + 1;                              // second run: [p_lo, p_hi)
            if (p_hi > P.nbase) p_hi = P.nbase;                                                  // partner of pair 0 is view 0 itself
            if (p_lo < a_hi) p_lo = a_hi;                                                        // the middle view, already sent
            if (p_hi > p_lo)
                CBCT_COMM(cm->broadcast(cm->ctx, (char *)L.d_T + (size_t)p_lo * per_base, (unsigned long long)(p_hi - p_lo) * per_base, r, st));
        }
    }
    CBCT_COMM(cm->allreduce_sum_f64(cm->ctx, g->d_partials, (unsigned long long)nblk, st));
    finalize_sums_kernel<<<1, 256, 0, st>>>(g->d_partials, (int)nblk, 1, g->partials_stride, d_sum_sq);
    CBCT_LAUNCH_CHECK(g);
    return CBCT_OK;
}

// d_g = f - coef P^T T on every rank
cbct_status sharded_back(const cbct_geometry *g, const Level &L, const cbct_comm *cm, const float *f, float coef, float *d_g,
                         cudaStream_t st)
{
    const LevelParams &P = L.p;
    cbct_status s;
    const int nzu = back_nzunits(L), unit = back_zunit(L), nzh = P.nz / P.nmir;
    Shard sh = {0, 0, 0, 0};
    shard_range(nzu, cm->world, cm->rank, &sh.zu_lo, &sh.zu_hi);
    if ((s = launch_back(g, L, L.d_T, 1, f, coef, d_g, st, &sh)) != CBCT_OK) return s;
    const size_t slice = (size_t)P.nx * P.ny * sizeof(float);
    for (int r = 0; r < cm->world; ++r) {
        int lo, hi;
        shard_range(nzu, cm->world, r, &lo, &hi);
        const int k_lo = lo * unit, k_hi = hi * unit < nzh ? hi * unit : nzh;
        if (k_hi <= k_lo) continue;
        CBCT_COMM(cm->broadcast(cm->ctx, (char *)d_g + (size_t)k_lo * slice, (unsigned long long)(k_hi - k_lo) * slice, r, st));
        if (P.nmir == 2)        // the mirror images of those slices
            CBCT_COMM(cm->broadcast(cm->ctx, (char *)d_g + (size_t)(P.nz - k_hi) * slice, (unsigned long long)(k_hi - k_lo) * slice, r, st));
    }
    return CBCT_OK;
}

// The whole reconstruction on device buffers (level-0 sized d_y, d_vol).  cm == NULL: one GPU.
cbct_status fbs_device(const cbct_geometry *g, const float *d_y, float *d_vol, const cbct_fbs_params *p,
                       cbct_fbs_report *rep, cudaStream_t st, const cbct_comm *cm = nullptr)
{
    cbct_status s;
    const int nl = p->n_levels;
    const bool want_obj = rep && rep->objective;
    {   // the objective monitor keeps one (E1, E2) pair per iteration on the device: its capacity bounds monitored calls only
        long total = 0;
        for (int l = 0; l < nl; ++l) total += p->iters_per_level[l];
        if (want_obj && total > g->objective_cap)
            return cbct_fail(CBCT_ERR_INVALID_ARG, "cbct_fbs_reconstruct: more than %d iterations in one call with the "
                             "objective monitor on (report->objective != NULL)", g->objective_cap);
    }
    // slot of iteration n's (E1, E2) pair: its own when monitored, else two scratch pairs taken in turn (the next
    // iteration's forward projection may be queued while this one's pair is still unread)
    auto obj_slot = [&](int n) { return g->d_objective + 2 * (want_obj ? n : (n & 1)); };
    CBCT_CUDA(cudaEventRecord(g->ev[0], st));
    if (!g->host_armijo)        // the cooperative TV-prox kernel counts its descent steps and trials on the device
        CBCT_CUDA(cudaMemsetAsync(g->d_scalars + 20, 0, 2 * sizeof(double), st));

    // data pyramid: y_l = 2x2 mean of y_{l-1}  (S12)
    {
        for (int l = 1; l < nl; ++l) {
            const float *src = (l == 1) ? d_y : g->levels[l - 1].d_y;
            if ((s = launch_bin(g, g->levels[l - 1], src, g->levels[l].d_y, st)) != CBCT_OK) return s;
        }
        // initial volume on the coarsest level
        if (p->use_initial) {
            for (int l = 1; l < nl; ++l) {
                const float *src = (l == 1) ? d_vol : g->levels[l - 1].d_f;
                if ((s = launch_restrict(g, g->levels[l - 1], src, g->levels[l].d_f, st)) != CBCT_OK) return s;
            }
        } else {
            float *dst = (nl == 1) ? d_vol : g->levels[nl - 1].d_f;
            if ((s = launch_fill(g, dst, g->levels[nl - 1].nvox, 0.0f, st)) != CBCT_OK) return s;
        }
    }

    const bool eq6 = p->backprojector == CBCT_BACKPROJECTOR_EQ6;
    int done = 0, inner_total = 0, trials_total = 0;
    int iters_done[8] = {0, 0, 0, 0, 0, 0, 0, 0};      // per level, coarsest -> finest (max_levels <= 8)
    for (int l = nl - 1; l >= 0; --l) {
        const Level &L = g->levels[l];
        float *f = (l == 0) ? d_vol : L.d_f;
        const float *y = (l == 0) ? d_y : L.d_y;
        const int n_it = p->iters_per_level[nl - 1 - l];
        double lhat = 0.0;
        {
            if ((s = step_bound_level(g, L, &lhat, st)) != CBCT_OK) return s;
        }
        if (!(lhat > 0.0)) return cbct_fail(CBCT_ERR_GEOMETRY, "level %d: no ray crosses the volume (Lhat = %g)", l, lhat);
        const double c_norm = 2.0 * (double)L.nvox / (double)L.nray;
        const double tau = p->step / lhat, w = tau * p->tv_weight;
        if (rep && rep->step_abs) rep->step_abs[nl - 1 - l] = tau;
        int it_done = 0;
        bool fwd_queued = false;        // this iteration's forward projection was queued by the previous one
        for (int it = 0; it < n_it; ++it, ++done) {
            if (p->conv_tol > 0.0)      // keep the volume that enters the iteration for the convergence test
                CBCT_CUDA(cudaMemcpyAsync(L.d_prev, f, L.nvox * sizeof(float), cudaMemcpyDeviceToDevice, st));
            if (cm) {
                if ((s = sharded_forward(g, L, cm, f, y, obj_slot(done) + 1, st)) != CBCT_OK) return s;
            } else if (!fwd_queued) {
                if ((s = launch_forward(g, L, f, y, L.d_T, eq6 ? 4 : 1, obj_slot(done) + 1, st)) != CBCT_OK) return s;
            }
            fwd_queued = false;
            if (want_obj) {
                if ((s = launch_tv_energy(g, L, f, p->tv.eps_delta, obj_slot(done), st)) != CBCT_OK) return s;
            }
            {
                if (cm) s = sharded_back(g, L, cm, f, (float)(tau * c_norm), L.d_g, st);
                else if (eq6) s = launch_back_eq6(g, L, L.d_T, f, (float)(tau * c_norm), L.d_g, st);
                else s = launch_back(g, L, L.d_T, 1, f, (float)(tau * c_norm), L.d_g, st);
                if (s != CBCT_OK) return s;
            }
            {
                cbct_tv_report tr;
                ForwardAhead fa = {g, &L, f, y, eq6 ? 4 : 1, obj_slot(done + 1) + 1, st};
                TvAhead ah = {forward_ahead, &fa, false};
                // (host-sequenced Armijo loop only: the cooperative kernel has no host wait to hide)
                const bool look_ahead = !cm && g->host_armijo && !want_obj && p->conv_tol == 0.0 && it + 1 < n_it;
                if ((s = run_tv_prox(g, L, L.d_g, f, w, p->nonneg, p->tv, &tr, false, st, look_ahead ? &ah : nullptr)) != CBCT_OK) return s;
                fwd_queued = look_ahead && ah.valid;
                inner_total += tr.inner_iters;
                trials_total += tr.trials;
            }
            ++it_done;
            if (p->conv_tol > 0.0) {    // "until convergence" (L145; reading S20): relative change of the volume
                double d2 = 0.0, p2 = 0.0;
                if ((s = volume_change(g, L.nvox, f, L.d_prev, &d2, &p2, st)) != CBCT_OK) return s;
                if (p2 > 0.0 && d2 <= p->conv_tol * p->conv_tol * p2) { ++done; break; }
            }
        }
        iters_done[nl - 1 - l] = it_done;
        if (rep && rep->iters_done) rep->iters_done[nl - 1 - l] = it_done;
        if (l > 0) {
            float *fine = (l == 1) ? d_vol : g->levels[l - 1].d_f;
            if ((s = launch_prolong(g, g->levels[l - 1], L.d_f, fine, st)) != CBCT_OK) return s;
        }
    }
    CBCT_CUDA(cudaEventRecord(g->ev[1], st));
    if (rep) {
        if (!g->host_armijo) CBCT_CUDA(cudaMemcpyAsync(g->h_scalars + 20, g->d_scalars + 20, 2 * sizeof(double), cudaMemcpyDeviceToHost, st));
        CBCT_CUDA(cudaStreamSynchronize(st));
        if (!g->host_armijo) { inner_total = (int)(g->h_scalars[20] + 0.5); trials_total = (int)(g->h_scalars[21] + 0.5); }
        rep->n_iters_total = done;
        rep->inner_total = inner_total;
        rep->trials_total = trials_total;
        CBCT_CUDA(cudaEventElapsedTime(&rep->ms_total, g->ev[0], g->ev[1]));
        if (want_obj && done > 0) {
            std::vector<double> h(2 * (size_t)done);
            CBCT_CUDA(cudaMemcpyAsync(h.data(), g->d_objective, sizeof(double) * 2 * done, cudaMemcpyDeviceToHost, st));
            CBCT_CUDA(cudaStreamSynchronize(st));
            int idx = 0;
            for (int l = nl - 1; l >= 0; --l) {
                const Level &L = g->levels[l];
                for (int it = 0; it < iters_done[nl - 1 - l]; ++it, ++idx)
                    rep->objective[idx] = p->tv_weight * h[2 * idx] / (double)L.nvox + h[2 * idx + 1] / (double)L.nray;
            }
        }
    }
    return CBCT_OK;
}

}  // namespace

extern "C" cbct_status cbct_step_bound(const cbct_geometry *g, int level, double *lhat, void *cuda_stream)
{
    const Level *L = get_level(g, level);
    if (!L || !lhat) return cbct_fail(CBCT_ERR_INVALID_ARG, "cbct_step_bound: bad handle, level or NULL");
    return step_bound_level(g, *L, lhat, (cudaStream_t)cuda_stream);
}

extern "C" cbct_status cbct_fbs_reconstruct(const cbct_geometry *g, const float *d_proj_y, float *d_vol_inout,
                                            const cbct_fbs_params *params, cbct_fbs_report *report,
                                            void *cuda_stream)
{
    cbct_status s = check_params(g, params);
    if (s != CBCT_OK) return s;
    if (!d_proj_y || !d_vol_inout) return cbct_fail(CBCT_ERR_INVALID_ARG, "cbct_fbs_reconstruct: NULL buffer");
    return fbs_device(g, d_proj_y, d_vol_inout, params, report, (cudaStream_t)cuda_stream);
}

extern "C" cbct_status cbct_shard_range(int n_units, int world, int rank, int *lo, int *hi)
{
    if (n_units < 0 || world < 1 || rank < 0 || rank >= world || !lo || !hi)
        return cbct_fail(CBCT_ERR_INVALID_ARG, "cbct_shard_range: bad argument");
    shard_range(n_units, world, rank, lo, hi);
    return CBCT_OK;
}

extern "C" cbct_status cbct_shard_units(const cbct_geometry *g, int level, int *n_base_views, int *n_z_units, int *z_unit_slices)
{
    const Level *L = get_level(g, level);
    if (!L) return cbct_fail(CBCT_ERR_INVALID_ARG, "cbct_shard_units: bad handle or level");
    if (n_base_views) *n_base_views = forward_units(*L);
    if (n_z_units) *n_z_units = back_nzunits(*L);
    if (z_unit_slices) *z_unit_slices = back_zunit(*L);
    return CBCT_OK;
}

extern "C" cbct_status cbct_fbs_reconstruct_sharded(const cbct_geometry *g, const cbct_comm *comm, const float *d_proj_y,
                                                    float *d_vol_inout, const cbct_fbs_params *params,
                                                    cbct_fbs_report *report, void *cuda_stream)
{
    cbct_status s = check_params(g, params);
    if (s != CBCT_OK) return s;
    if (!d_proj_y || !d_vol_inout) return cbct_fail(CBCT_ERR_INVALID_ARG, "cbct_fbs_reconstruct_sharded: NULL buffer");
    if (!comm || comm->world < 1 || comm->rank < 0 || comm->rank >= comm->world || !comm->broadcast || !comm->allreduce_sum_f64)
        return cbct_fail(CBCT_ERR_INVALID_ARG, "cbct_fbs_reconstruct_sharded: bad communicator");
    if (params->backprojector != CBCT_BACKPROJECTOR_EXACT)
        return cbct_fail(CBCT_ERR_UNSUPPORTED, "cbct_fbs_reconstruct_sharded: only the exact-transpose back-projector is sharded");
    return fbs_device(g, d_proj_y, d_vol_inout, params, report, (cudaStream_t)cuda_stream, comm);
}

extern "C" cbct_status cbct_fbs_reconstruct_host(const cbct_geometry *g, const float *h_proj_y,
                                                 float *h_vol_inout, const cbct_fbs_params *params,
                                                 cbct_fbs_report *report, void *cuda_stream)
{
    cbct_status s = check_params(g, params);
    if (s != CBCT_OK) return s;
    if (!h_proj_y || !h_vol_inout) return cbct_fail(CBCT_ERR_INVALID_ARG, "cbct_fbs_reconstruct_host: NULL buffer");
    cudaStream_t st = (cudaStream_t)cuda_stream;
    const Level &L0 = g->levels[0];
    CBCT_CUDA(cudaMemcpyAsync(L0.d_y, h_proj_y, L0.nray * sizeof(float), cudaMemcpyHostToDevice, st));
    if (params->use_initial)
        CBCT_CUDA(cudaMemcpyAsync(L0.d_f, h_vol_inout, L0.nvox * sizeof(float), cudaMemcpyHostToDevice, st));
    s = fbs_device(g, L0.d_y, L0.d_f, params, report, st);
    if (s != CBCT_OK) return s;
    CBCT_CUDA(cudaMemcpyAsync(h_vol_inout, L0.d_f, L0.nvox * sizeof(float), cudaMemcpyDeviceToHost, st));
    CBCT_CUDA(cudaStreamSynchronize(st));
    return CBCT_OK;
}
