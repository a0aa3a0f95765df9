// solve.inl -- the Born-term loop and its drivers (included at the end of tbs.cu).

namespace {

// Build (once) a CUDA graph holding `batch` terms for frequency f.
tbs_status build_graph(tbs_plan *pl, Freq &f, int batch, cudaStream_t st) {
    if (f.graph && f.graph_batch == batch) return TBS_OK;
    if (f.graph) { cudaGraphExecDestroy(f.graph); f.graph = nullptr; }
    cudaStream_t cs;
    CU(pl, cudaStreamCreateWithFlags(&cs, cudaStreamNonBlocking));
    cudaGraph_t g = nullptr;
    cudaError_t e = cudaStreamBeginCapture(cs, cudaStreamCaptureModeThreadLocal);
    if (e == cudaSuccess) {
        for (int i = 0; i < batch && e == cudaSuccess; ++i) e = launch_term(pl, f, cs);
        cudaError_t e2 = cudaStreamEndCapture(cs, &g);
        if (e == cudaSuccess) e = e2;
    }
    if (e == cudaSuccess) e = cudaGraphInstantiate(&f.graph, g, 0);
    if (g) cudaGraphDestroy(g);
    cudaStreamDestroy(cs);
    (void)st;
    if (e != cudaSuccess) { f.graph = nullptr; return fail(pl, TBS_ERR_CUDA, "graph build: %s", cudaGetErrorString(e)); }
    f.graph_batch = batch;
    return TBS_OK;
}

// Run the series for one frequency.  The field is left in f.p, history in pl->h_hist.
tbs_status solve_one(tbs_plan *pl, int ifreq, int max_terms, double tol, cudaStream_t st, int *n_terms_out) {
    Freq &f = pl->fr[ifreq];
    if (!f.have_V) return fail(pl, TBS_ERR_NOT_READY, "tbs_set_medium / tbs_set_potential not called");
    if (!f.have_S) return fail(pl, TBS_ERR_NOT_READY, "tbs_set_source / tbs_set_source_field not called");
    tbs_status hs = ensure_history(pl, max_terms);
    if (hs != TBS_OK) return hs;
    const int batch = pl->graph_batch > 0 ? pl->graph_batch : 8;
    if (pl->graph_batch > 0) {
        tbs_status gs = build_graph(pl, f, batch, st);
        if (gs != TBS_OK) return gs;
    }
    Ctl *h = pl->h_ctl;
    memset(&h[0], 0, sizeof(Ctl));
    h[0].max_terms = max_terms;
    h[0].tol = tol;
    h[0].status = 1;
    CU(pl, cudaMemcpyAsync(f.ctl, &h[0], sizeof(Ctl), cudaMemcpyHostToDevice, st));
    CU(pl, cudaMemsetAsync(pl->norms, 0, sizeof(double) * 2 * (max_terms + 1), st));
    CU(pl, cudaMemsetAsync(pl->history, 0, sizeof(double) * (max_terms + 1), st));
    CU(pl, cudaEventRecord(pl->ev_t0, st));
    // term 0 forward half: W = FFT_x(pad(S / k0^2))
    RowArgs r;
    fill_row_args(pl, f, r, f.S, (float)(1.0 / (f.k0 * f.k0)), 1);
    CU(pl, launch_row<true>(pl->n[0], r, st));
    pl->launches += 1;
    const int per_term = mid_launches(pl) + 1;
    // batches, double-buffered: enqueue batch i+1 before looking at the flag of batch i
    int issued = 0;
    bool done = false;
    const int max_batches = (max_terms + 1 + batch - 1) / batch + 1;
    for (int b = 0; b < max_batches + 1 && !done; ++b) {
        if (b < max_batches) {
            if (pl->graph_batch > 0) {
                CU(pl, cudaGraphLaunch(f.graph, st));
            } else {
                for (int i = 0; i < batch; ++i) CU(pl, launch_term(pl, f, st));
            }
            pl->launches += (long long)batch * per_term;
            CU(pl, cudaMemcpyAsync(&h[1 + (b & 1)], f.ctl, sizeof(Ctl), cudaMemcpyDeviceToHost, st));
            CU(pl, cudaEventRecord(pl->ev[b & 1], st));
            ++issued;
        }
        if (b >= 1) {
            CU(pl, cudaEventSynchronize(pl->ev[(b - 1) & 1]));
            if (h[1 + ((b - 1) & 1)].done) done = true;
        }
    }
    CU(pl, cudaEventRecord(pl->ev_t1, st));
    CU(pl, cudaMemcpyAsync(&h[3], f.ctl, sizeof(Ctl), cudaMemcpyDeviceToHost, st));
    CU(pl, cudaMemcpyAsync(pl->h_hist, pl->history, sizeof(double) * (max_terms + 1), cudaMemcpyDeviceToHost, st));
    CU(pl, cudaStreamSynchronize(st));
    float ms = 0.f;
    cudaEventElapsedTime(&ms, pl->ev_t0, pl->ev_t1);
    pl->loop_ms += ms;
    if (!h[3].done) return fail(pl, TBS_ERR_CUDA, "term loop ended without the stop flag (issued %d batches)", issued);
    *n_terms_out = h[3].n_terms;
    if (h[3].status == TBS_ERR_DIVERGED) fail(pl, TBS_ERR_DIVERGED, "term norm became non-finite at term %d", h[3].n_terms);
    return (tbs_status)h[3].status;
}

tbs_status worst(tbs_status a, tbs_status b) {
    if (a < 0) return a;
    if (b < 0) return b;
    return a > b ? a : b;
}

tbs_status solve_all(tbs_plan *pl, int max_terms, double tol, float *p_out, bool out_is_host,
                     double *history, int32_t *n_terms, cudaStream_t st) {
    if (!pl || max_terms < 0 || !(tol >= 0) || !p_out || !history || !n_terms) return TBS_ERR_INVALID_ARG;
    pl->launches = 0;
    pl->loop_ms = 0;
    tbs_status res = TBS_OK;
    for (int i = 0; i < (int)pl->fr.size(); ++i) {
        int nt = 0;
        tbs_status s = solve_one(pl, i, max_terms, tol, st, &nt);
        if (s < 0 && s != TBS_ERR_DIVERGED) return s;
        n_terms[i] = nt;
        double *hrow = history + (size_t)i * (max_terms + 1);
        for (int k = 0; k <= max_terms; ++k) hrow[k] = k <= nt ? pl->h_hist[k] : 0.0;
        CU(pl, cudaMemcpyAsync((float2 *)p_out + (size_t)i * pl->npts, pl->fr[i].p, sizeof(float2) * pl->npts,
                               out_is_host ? cudaMemcpyDeviceToHost : cudaMemcpyDeviceToDevice, st));
        res = worst(res, s);
    }
    CU(pl, cudaStreamSynchronize(st));
    return res;
}

}  // namespace

extern "C" {

tbs_status tbs_solve(tbs_plan *pl, int max_terms, double tol, float *p_out, double *history,
                     int32_t *n_terms, void *stream) {
    return solve_all(pl, max_terms, tol, p_out, false, history, n_terms, (cudaStream_t)stream);
}

tbs_status tbs_solve_host(tbs_plan *pl, int max_terms, double tol, float *p_out_host, double *history,
                          int32_t *n_terms, void *stream) {
    return solve_all(pl, max_terms, tol, p_out_host, true, history, n_terms, (cudaStream_t)stream);
}

tbs_status tbs_apply_green(tbs_plan *pl, int ifreq, const float *x, float *out, void *stream) {
    if (!pl || !x || !out || ifreq < 0 || ifreq >= (int)pl->fr.size()) return TBS_ERR_INVALID_ARG;
    cudaStream_t st = (cudaStream_t)stream;
    Freq &f = pl->fr[ifreq];
    tbs_status hs = ensure_history(pl, 1);
    if (hs != TBS_OK) return hs;
    // Save the plan's running field: the inverse half writes p.
    Ctl *h = pl->h_ctl;
    memset(&h[0], 0, sizeof(Ctl));
    h[0].max_terms = 1 << 30;
    h[0].tol = 0.0;
    CU(pl, cudaMemcpyAsync(f.ctl, &h[0], sizeof(Ctl), cudaMemcpyHostToDevice, st));
    CU(pl, cudaMemsetAsync(pl->norms, 0, sizeof(double) * 2 * pl->hist_cap, st));
    // Use `out` itself as the field buffer and a unit window-free pass: A is applied (as in u_0).
    RowArgs r;
    fill_row_args(pl, f, r, (const float2 *)x, (float)(1.0 / (f.k0 * f.k0)), 1);
    CU(pl, launch_row<true>(pl->n[0], r, st));
    CU(pl, launch_mid_passes(pl, f, st));
    fill_row_args(pl, f, r, nullptr, 0.f, 0);
    r.ucbs = nullptr;  // one plain application of G, whatever the plan's scheme
    r.p = (float2 *)out;
    r.V = f.V;  // only multiplies a value that is dropped when do_fwd = 0
    CU(pl, launch_row<false>(pl->n[0], r, st));
    CU(pl, cudaStreamSynchronize(st));
    return TBS_OK;
}

tbs_status tbs_solve_harmonics(tbs_plan *const *plans, int n_harm, int max_terms, double tol, int ref_row,
                               double surface_pressure_pa, float *const *p_out, double *const *history,
                               int32_t *n_terms, void *stream) {
    if (!plans || n_harm < 1 || n_harm > 5 || !p_out || !history || !n_terms) return TBS_ERR_INVALID_ARG;
    for (int h = 0; h < n_harm; ++h)
        if (!plans[h] || !p_out[h] || !history[h] || plans[h]->fr.size() != 1) return TBS_ERR_INVALID_ARG;
    tbs_plan *p1 = plans[0];
    for (int h = 1; h < n_harm; ++h) {
        tbs_plan *ph = plans[h];
        if (ph->ndim != p1->ndim) return fail(ph, TBS_ERR_INVALID_ARG, "plans differ in dimension");
        for (int a = 0; a < 3; ++a)
            if (p1->n[a] != ph->n[a]) return fail(ph, TBS_ERR_INVALID_ARG, "plans differ in grid size");
        if (fabs(ph->fr[0].f - (h + 1) * p1->fr[0].f) > 1e-9 * p1->fr[0].f)
            return fail(ph, TBS_ERR_INVALID_ARG, "plan %d must be created at %d times the fundamental", h, h + 1);
    }
    const int nslow = p1->ndim == 2 ? p1->n[1] : p1->n[2];
    if (ref_row < 0 || ref_row >= nslow) return fail(p1, TBS_ERR_INVALID_ARG, "ref_row outside the grid");
    cudaStream_t st = (cudaStream_t)stream;
    const long long n = p1->npts;
    tbs_status res = solve_all(p1, max_terms, tol, p_out[0], false, history[0], &n_terms[0], st);
    if (res < 0) return res;
    if (surface_pressure_pa > 0.0) {
        const long long slab = n / nslow;
        cudaMemsetAsync(p1->maxbits, 0, sizeof(unsigned int), st);
        k_row_max<<<nblk(slab, 256), 256, 0, st>>>(p1->fr[0].p, (long long)ref_row * slab, slab, p1->maxbits);
        k_rescale_field<<<nblk(n, 256), 256, 0, st>>>(p1->fr[0].p, p1->maxbits, surface_pressure_pa, n);
        CU(p1, cudaGetLastError());
        CU(p1, cudaMemcpyAsync(p_out[0], p1->fr[0].p, sizeof(float2) * n, cudaMemcpyDeviceToDevice, st));
        p1->launches += 2;
    }
    // xi = beta/(rho0 c0^4); S_h = -xi (h w1)^2 C_h (Eqs. 28b-28e)
    const double xi = p1->beta / (p1->rho0 * pow(p1->c0, 4.0));
    for (int h = 2; h <= n_harm; ++h) {
        tbs_plan *ph = plans[h - 1];
        const double wh = (double)h * p1->fr[0].omega;
        const double coef = -xi * wh * wh;
        const float2 *f1 = plans[0]->fr[0].p;
        const float2 *f2 = h >= 3 ? plans[1]->fr[0].p : nullptr;
        const float2 *f3 = h >= 4 ? plans[2]->fr[0].p : nullptr;
        const float2 *f4 = h >= 5 ? plans[3]->fr[0].p : nullptr;
        float2 *S = ph->fr[0].S;
        const unsigned g = nblk(n, 256);
        if (h == 2) k_harmonic_source<<<g, 256, 0, st>>>(S, coef, f1, f1, 0.5, nullptr, nullptr, 0.0, n);
        else if (h == 3) k_harmonic_source<<<g, 256, 0, st>>>(S, coef, f1, f2, 1.0, nullptr, nullptr, 0.0, n);
        else if (h == 4) k_harmonic_source<<<g, 256, 0, st>>>(S, coef, f2, f2, 0.5, f1, f3, 1.0, n);
        else k_harmonic_source<<<g, 256, 0, st>>>(S, coef, f2, f3, 1.0, f1, f4, 1.0, n);
        CU(ph, cudaGetLastError());
        ph->fr[0].have_S = true;
        tbs_status sh = solve_all(ph, max_terms, tol, p_out[h - 1], false, history[h - 1], &n_terms[h - 1], st);
        ph->launches += 1;
        if (sh < 0) return sh;
        res = worst(res, sh);
    }
    return res;
}

tbs_status tbs_solve_second_harmonic(tbs_plan *p1, tbs_plan *p2, int max_terms, double tol, int ref_row,
                                     double surface_pressure_pa, float *p1_out, float *p2_out,
                                     double *history1, double *history2, int32_t *n_terms1,
                                     int32_t *n_terms2, void *stream) {
    if (!n_terms1 || !n_terms2) return TBS_ERR_INVALID_ARG;
    tbs_plan *plans[2] = {p1, p2};
    float *outs[2] = {p1_out, p2_out};
    double *hist[2] = {history1, history2};
    int32_t nt[2] = {0, 0};
    const tbs_status s = tbs_solve_harmonics(plans, 2, max_terms, tol, ref_row, surface_pressure_pa, outs, hist, nt, stream);
    *n_terms1 = nt[0];
    *n_terms2 = nt[1];
    return s;
}

tbs_status tbs_profile_term(tbs_plan *pl, int ifreq, int reps, double out_ms[4], void *stream) {
    if (!pl || !out_ms || reps < 1 || reps > 256 || ifreq < 0 || ifreq >= (int)pl->fr.size()) return TBS_ERR_INVALID_ARG;
    Freq &f = pl->fr[ifreq];
    if (!f.have_V || !f.have_S) return fail(pl, TBS_ERR_NOT_READY, "medium and source required");
    cudaStream_t st = (cudaStream_t)stream;
    tbs_status hs = ensure_history(pl, reps + 4);
    if (hs != TBS_OK) return hs;
    // A real series: term 0, two warm-up terms, then `reps` terms with an event between kernels.
    Ctl *h = pl->h_ctl;
    memset(&h[0], 0, sizeof(Ctl));
    h[0].max_terms = 1 << 30;
    h[0].tol = 0.0;
    CU(pl, cudaMemcpyAsync(f.ctl, &h[0], sizeof(Ctl), cudaMemcpyHostToDevice, st));
    CU(pl, cudaMemsetAsync(pl->norms, 0, sizeof(double) * 2 * pl->hist_cap, st));
    RowArgs r;
    fill_row_args(pl, f, r, f.S, (float)(1.0 / (f.k0 * f.k0)), 1);
    CU(pl, launch_row<true>(pl->n[0], r, st));
    for (int i = 0; i < 3; ++i) CU(pl, launch_term(pl, f, st));
    const int nmid = mid_launches(pl);
    const int per = nmid + 1;
    std::vector<cudaEvent_t> evs((size_t)reps * per + 1);
    for (auto &e : evs) CU(pl, cudaEventCreate(&e));
    fill_row_args(pl, f, r, nullptr, 0.f, 1);
    CU(pl, cudaEventRecord(evs[0], st));
    for (int i = 0; i < reps; ++i) {
        for (int k = 0; k < nmid; ++k) {
            CU(pl, launch_mid_passes(pl, f, st, k));
            CU(pl, cudaEventRecord(evs[(size_t)i * per + k + 1], st));
        }
        CU(pl, launch_row<false>(pl->n[0], r, st));
        CU(pl, cudaEventRecord(evs[(size_t)i * per + nmid + 1], st));
    }
    CU(pl, cudaStreamSynchronize(st));
    for (int k = 0; k < 4; ++k) out_ms[k] = 0.0;
    for (int i = 0; i < reps; ++i)
        for (int k = 0; k < per; ++k) {
            float ms = 0.f;
            cudaEventElapsedTime(&ms, evs[(size_t)i * per + k], evs[(size_t)i * per + k + 1]);
            // out_ms[0] = row kernel, out_ms[1..] = column/plane passes in launch order
            out_ms[k == nmid ? 0 : k + 1] += ms / reps;
        }
    for (auto &e : evs) cudaEventDestroy(e);
    return TBS_OK;
}

}  // extern "C"
