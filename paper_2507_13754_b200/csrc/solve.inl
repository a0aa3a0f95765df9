// solve.inl -- the Born-term loop and its drivers (included at the end of tbs.cu).

namespace {

// Build (once) a CUDA graph holding `batch` terms of frequency f on slot `si`; half = 1: grids sized for half of
// the SMs (two members of a frequency batch share the GPU).
tbs_status build_graph(tbs_plan *pl, Freq &f, int si, int half, int batch) {
    TermGraph &tg = f.graph[si][half];
    if (tg.exec && tg.batch == batch) return TBS_OK;
    if (tg.exec) { cudaGraphExecDestroy(tg.exec); tg.exec = nullptr; }
    cudaStream_t cs;
    CU(pl, cudaStreamCreateWithFlags(&cs, cudaStreamNonBlocking));
    cudaGraph_t g = nullptr;
    LaunchOpt opt;
    opt.sm_limit = half ? (pl->sms + 1) / 2 : 0;
    opt.overlap = pl->overlap != 0;
    cudaError_t e = cudaStreamBeginCapture(cs, cudaStreamCaptureModeThreadLocal);
    if (e == cudaSuccess) {
        for (int i = 0; i < batch && e == cudaSuccess; ++i) e = launch_term(pl, f, pl->slot[si], cs, opt);
        cudaError_t e2 = cudaStreamEndCapture(cs, &g);
        if (e == cudaSuccess) e = e2;
    }
    if (e == cudaSuccess) e = cudaGraphInstantiate(&tg.exec, g, 0);
    if (g) cudaGraphDestroy(g);
    cudaStreamDestroy(cs);
    if (e != cudaSuccess) { tg.exec = nullptr; return fail(pl, TBS_ERR_CUDA, "graph build: %s", cudaGetErrorString(e)); }
    tg.batch = batch;
    return TBS_OK;
}

// One series in flight on a slot: term 0, then batches of terms with the stop flag read back double-buffered
// (batch i+1 is enqueued before the flag of batch i is looked at).
struct Run {
    int ifreq = -1;
    int si = 0;
    cudaStream_t st = nullptr;
    int half = 0;
    int issued = 0;      // batches enqueued
    int checked = 0;     // batches whose flag has been read
    int max_batches = 0;
    bool active = false;
};

tbs_status run_begin(tbs_plan *pl, Run &r, int ifreq, int si, cudaStream_t st, int half, int max_terms, double tol,
                     bool resume = false) {
    Freq &f = pl->fr[ifreq];
    Slot &s = pl->slot[si];
    if (!f.have_V) return fail(pl, TBS_ERR_NOT_READY, "tbs_set_medium / tbs_set_potential not called");
    if (!f.have_S) return fail(pl, TBS_ERR_NOT_READY, "tbs_set_source / tbs_set_source_field not called");
    const int batch = pl->graph_batch > 0 ? pl->graph_batch : 8;
    r = Run();
    r.ifreq = ifreq; r.si = si; r.st = st; r.half = half; r.active = true;
    r.max_batches = (max_terms + 1 + batch - 1) / batch + 1;
    Ctl *h = s.h_ctl;
    if (resume) {
        // tbs_solve_resume: the series stopped at its cap with W1 holding the forward half of the next term, p the
        // partial sum and norms / history the terms so far: lift the cap and go on from the term counter
        CU(pl, cudaMemcpyAsync(&h[0], f.ctl, sizeof(Ctl), cudaMemcpyDeviceToHost, st));
        CU(pl, cudaStreamSynchronize(st));
        if (!h[0].done || h[0].status != TBS_NOT_CONVERGED) return fail(pl, TBS_ERR_NOT_READY, "no capped series to resume");
        if (max_terms <= h[0].n_terms) return fail(pl, TBS_ERR_INVALID_ARG, "max_terms must exceed the %d terms already summed", h[0].n_terms);
        r.max_batches = (max_terms - h[0].n_terms + batch - 1) / batch + 1;
        h[0].done = 0;
        h[0].max_terms = max_terms;
        h[0].tol = tol;
        h[0].status = 1;
        CU(pl, cudaMemcpyAsync(f.ctl, &h[0], sizeof(Ctl), cudaMemcpyHostToDevice, st));
        CU(pl, cudaEventRecord(s.ev_t0, st));
        return TBS_OK;
    }
    memset(&h[0], 0, sizeof(Ctl));
    h[0].max_terms = max_terms;
    h[0].tol = tol;
    h[0].status = 1;
    CU(pl, cudaMemcpyAsync(f.ctl, &h[0], sizeof(Ctl), cudaMemcpyHostToDevice, st));
    CU(pl, cudaMemsetAsync(s.norms, 0, sizeof(double) * 2 * (max_terms + 1), st));
    CU(pl, cudaMemsetAsync(s.history, 0, sizeof(double) * (max_terms + 1), st));
    CU(pl, cudaEventRecord(s.ev_t0, st));
    // term 0 forward half: W = FFT_x(pad(S / k0^2))
    RowArgs ra;
    fill_row_args(pl, f, s, ra, f.S, (float)(1.0 / (f.k0 * f.k0)), 1);
    LaunchOpt opt;
    opt.sm_limit = half ? (pl->sms + 1) / 2 : 0;
    CU(pl, launch_row(pl->n[0], true, ra, st, false, opt));
    pl->launches += 1;
    return TBS_OK;
}

// Enqueue one more batch of terms (and the read-back of the flag behind it).
tbs_status run_enqueue(tbs_plan *pl, Run &r) {
    Freq &f = pl->fr[r.ifreq];
    Slot &s = pl->slot[r.si];
    const int batch = pl->graph_batch > 0 ? pl->graph_batch : 8;
    if (pl->graph_batch > 0) {
        tbs_status gs = build_graph(pl, f, r.si, r.half, batch);
        if (gs != TBS_OK) return gs;
        CU(pl, cudaGraphLaunch(f.graph[r.si][r.half].exec, r.st));
    } else {
        LaunchOpt opt;
        opt.sm_limit = r.half ? (pl->sms + 1) / 2 : 0;
        opt.overlap = pl->overlap != 0;
        for (int i = 0; i < batch; ++i) CU(pl, launch_term(pl, f, s, r.st, opt));
    }
    pl->launches += (long long)batch * (mid_launches(pl) + 1);
    CU(pl, cudaMemcpyAsync(&s.h_ctl[1 + (r.issued & 1)], f.ctl, sizeof(Ctl), cudaMemcpyDeviceToHost, r.st));
    CU(pl, cudaEventRecord(s.ev[r.issued & 1], r.st));
    ++r.issued;
    return TBS_OK;
}

// Wait for the oldest unchecked batch; *done = its stop flag.
tbs_status run_check(tbs_plan *pl, Run &r, bool *done) {
    Slot &s = pl->slot[r.si];
    CU(pl, cudaEventSynchronize(s.ev[r.checked & 1]));
    *done = s.h_ctl[1 + (r.checked & 1)].done != 0;
    ++r.checked;
    return TBS_OK;
}

// The series has stopped: copy the field and the history out; the slot is free afterwards.
tbs_status run_finish(tbs_plan *pl, Run &r, int max_terms, float *p_out, bool out_is_host, double *history,
                      int32_t *n_terms, tbs_status *status) {
    Freq &f = pl->fr[r.ifreq];
    Slot &s = pl->slot[r.si];
    CU(pl, cudaEventRecord(s.ev_t1, r.st));
    CU(pl, cudaMemcpyAsync(&s.h_ctl[3], f.ctl, sizeof(Ctl), cudaMemcpyDeviceToHost, r.st));
    CU(pl, cudaMemcpyAsync(s.h_hist, s.history, sizeof(double) * (max_terms + 1), cudaMemcpyDeviceToHost, r.st));
    CU(pl, cudaMemcpyAsync((float2 *)p_out + (size_t)r.ifreq * pl->npts, f.p, sizeof(float2) * pl->npts,
                           out_is_host ? cudaMemcpyDeviceToHost : cudaMemcpyDeviceToDevice, r.st));
    CU(pl, cudaStreamSynchronize(r.st));
    r.active = false;
    const Ctl &c = s.h_ctl[3];
    if (!c.done) return fail(pl, TBS_ERR_CUDA, "term loop ended without the stop flag (issued %d batches)", r.issued);
    n_terms[r.ifreq] = c.n_terms;
    double *hrow = history + (size_t)r.ifreq * (max_terms + 1);
    for (int k = 0; k <= max_terms; ++k) hrow[k] = k <= c.n_terms ? s.h_hist[k] : 0.0;
    if (c.status == TBS_ERR_DIVERGED)
        fail(pl, TBS_ERR_DIVERGED, "series diverged at term %d of frequency %d (non-finite or growing term norm, PAPER.md:158)",
             c.n_terms, r.ifreq);
    *status = (tbs_status)c.status;
    return TBS_OK;
}

tbs_status worst(tbs_status a, tbs_status b) {
    if (a < 0) return a;
    if (b < 0) return b;
    return a > b ? a : b;
}

// All frequencies of the plan.  One frequency: the series runs on the caller's stream on slot 0.  Several: up to
// `concurrency` members are in flight at once, each on its slot's own stream, so that the HBM-bound passes of one
// member overlap the FP32-bound convolution pass of another; a member that has converged hands its slot to the
// next frequency.
constexpr bool kHalfWidthBatchGrids = false;
tbs_status solve_all(tbs_plan *pl, int max_terms, double tol, float *p_out, bool out_is_host,
                     double *history, int32_t *n_terms, cudaStream_t st, bool resume = false) {
    if (!pl || max_terms < 0 || !(tol >= 0) || !p_out || !history || !n_terms) return TBS_ERR_INVALID_ARG;
    if (resume && (pl->fr.size() != 1 || pl->resume_epoch != pl->epoch))
        return fail(pl, TBS_ERR_NOT_READY, "tbs_solve_resume: the last call was not a capped solve of this single-frequency plan");
    tbs_status ws = ensure_workspace(pl);
    if (ws != TBS_OK) return ws;
    pl->launches = 0;
    pl->loop_ms = 0;
    tbs_status hs = ensure_history(pl, max_terms, resume);
    if (hs != TBS_OK) return hs;
    pl->resume_epoch = ~0ull;
    const int nf = (int)pl->fr.size();
    const int conc = nf > 1 ? (pl->concurrency < pl->nslots ? pl->concurrency : pl->nslots) : 1;
    tbs_status res = TBS_OK;
    Run run[kMaxSlots];
    int next = 0, live = 0;
    const bool forked = conc > 1;
    CU(pl, cudaEventRecord(pl->ev_b0, st));
    if (forked) {
        CU(pl, cudaEventRecord(pl->ev_fork, st));
        for (int i = 0; i < conc; ++i) CU(pl, cudaStreamWaitEvent(pl->slot[i].own_stream, pl->ev_fork, 0));
    }
    auto start_next = [&](int si) -> tbs_status {
        if (next >= nf) return TBS_OK;
        // Grid width of members in flight together.  Measured on B200 (two members): full-width grids (the block
        // scheduler interleaves the two members' CTAs as SM resources free up) 9.97 -> 9.54 s on the 16-frequency
        // 256^3 batch and 126 -> 93 ms at 64^3; grids sized for half of the SMs each 9.70 -> 9.86 s and 126 -> 93 ms.
        const int half = kHalfWidthBatchGrids && forked && (live + 1 > 1 || nf - next > 1) ? 1 : 0;
        tbs_status s = run_begin(pl, run[si], next, si, forked ? pl->slot[si].own_stream : st, half, max_terms, tol, resume);
        if (s == TBS_OK) { ++next; ++live; }
        return s;
    };
    for (int i = 0; i < conc; ++i) {
        tbs_status s = start_next(i);
        if (s != TBS_OK) return s;
    }
    while (live > 0) {
        // keep two batches in flight on every live slot, then look at the oldest flag of each
        for (int i = 0; i < conc; ++i) {
            Run &r = run[i];
            while (r.active && r.issued - r.checked < 2 && r.issued < r.max_batches) {
                if (forked && live == 1 && next >= nf) r.half = 0;   // alone: full-width grids from here on
                tbs_status s = run_enqueue(pl, r);
                if (s != TBS_OK) return s;
            }
        }
        for (int i = 0; i < conc; ++i) {
            Run &r = run[i];
            if (!r.active) continue;
            if (r.checked >= r.issued) return fail(pl, TBS_ERR_CUDA, "term loop ran out of batches without the stop flag");
            bool done = false;
            tbs_status s = run_check(pl, r, &done);
            if (s != TBS_OK) return s;
            if (!done) continue;
            tbs_status sf = TBS_OK;
            s = run_finish(pl, r, max_terms, p_out, out_is_host, history, n_terms, &sf);
            if (s != TBS_OK) return s;
            --live;
            if (!forked) {
                float ms = 0.f;
                cudaEventElapsedTime(&ms, pl->slot[i].ev_t0, pl->slot[i].ev_t1);
                pl->loop_ms += ms;
            }
            if (sf < 0 && sf != TBS_ERR_DIVERGED) return sf;
            res = worst(res, sf);
            s = start_next(i);
            if (s != TBS_OK) return s;
        }
    }
    if (forked) {
        for (int i = 0; i < conc; ++i) {
            CU(pl, cudaEventRecord(pl->slot[i].ev_join, pl->slot[i].own_stream));
            CU(pl, cudaStreamWaitEvent(st, pl->slot[i].ev_join, 0));
        }
    }
    CU(pl, cudaEventRecord(pl->ev_b1, st));
    CU(pl, cudaStreamSynchronize(st));
    if (forked) {
        float ms = 0.f;
        cudaEventElapsedTime(&ms, pl->ev_b0, pl->ev_b1);
        pl->loop_ms = ms;   // members overlap: device time of the whole batch
    }
    if (nf == 1 && res == TBS_NOT_CONVERGED) pl->resume_epoch = pl->epoch;   // tbs_solve_resume may go on from here
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

tbs_status tbs_solve_resume(tbs_plan *pl, int max_terms, double tol, float *p_out, double *history,
                            int32_t *n_terms, void *stream) {
    return solve_all(pl, max_terms, tol, p_out, false, history, n_terms, (cudaStream_t)stream, true);
}

tbs_status tbs_apply_green(tbs_plan *pl, int ifreq, const float *x, float *out, void *stream) {
    if (pl) ++pl->epoch;
    if (!pl || !x || !out || ifreq < 0 || ifreq >= (int)pl->fr.size()) return TBS_ERR_INVALID_ARG;
    tbs_status ws = ensure_workspace(pl);
    if (ws != TBS_OK) return ws;
    cudaStream_t st = (cudaStream_t)stream;
    Freq &f = pl->fr[ifreq];
    Slot &s = pl->slot[0];
    tbs_status hs = ensure_history(pl, 1);
    if (hs != TBS_OK) return hs;
    Ctl *h = s.h_ctl;
    memset(&h[0], 0, sizeof(Ctl));
    h[0].max_terms = 1 << 30;
    h[0].tol = 0.0;
    h[0].hold = 1;
    CU(pl, cudaMemcpyAsync(f.ctl, &h[0], sizeof(Ctl), cudaMemcpyHostToDevice, st));
    CU(pl, cudaMemsetAsync(s.norms, 0, sizeof(double) * 2 * pl->hist_cap, st));
    // `out` itself serves as the field buffer of a window-carrying pass: A is applied (as in u_0).
    RowArgs r;
    fill_row_args(pl, f, s, r, (const float2 *)x, (float)(1.0 / (f.k0 * f.k0)), 1);
    CU(pl, launch_row(pl->n[0], true, r, st));
    KAbs keep = f.kabs;
    f.kabs = KAbs{0.f, 0.f, 0.f, 0.f};   // one plain application of G, whatever the plan's potential form
    cudaError_t e = launch_mid_passes(pl, f, s, st);
    f.kabs = keep;
    CU(pl, e);
    fill_row_args(pl, f, s, r, nullptr, 0.f, 0);
    r.ucbs = nullptr;  // ... and whatever the plan's scheme
    r.p = (float2 *)out;
    r.V = f.V;  // only multiplies a value that is dropped when do_fwd = 0
    CU(pl, launch_row(pl->n[0], false, r, st));
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
        tbs_status ws = ensure_workspace(ph);
        if (ws != TBS_OK) return ws;
    }
    const int nslow = p1->ndim == 2 ? p1->n[1] : p1->n[2];
    if (ref_row < 0 || ref_row >= nslow) return fail(p1, TBS_ERR_INVALID_ARG, "ref_row outside the grid");
    cudaStream_t st = (cudaStream_t)stream;
    const long long n = p1->npts;
    tbs_status res = solve_all(p1, max_terms, tol, p_out[0], false, history[0], &n_terms[0], st);
    if (res < 0) return res;
    if (surface_pressure_pa > 0.0) {
        const long long slab = n / nslow;
        CU(p1, cudaMemsetAsync(p1->maxbits, 0, sizeof(unsigned int), st));
        k_row_max<<<nblk(slab, 256), 256, 0, st>>>(p1->fr[0].p, (long long)ref_row * slab, slab, p1->maxbits);
        unsigned int bits = 0;
        CU(p1, cudaMemcpyAsync(&bits, p1->maxbits, sizeof bits, cudaMemcpyDeviceToHost, st));
        CU(p1, cudaStreamSynchronize(st));
        if (bits == 0u) return fail(p1, TBS_ERR_INVALID_ARG, "the fundamental vanishes on the reference row: nothing to rescale");
        ++p1->epoch;   // the running field no longer is the series' partial sum
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

// Per-kernel device time of one term.  Each kernel of the term is launched `reps` times back to back between two
// events on `stream` (so the events cost nothing per launch), after a live series of term 0 and three warm-up
// terms has put real data in place; the stop logic is held off (Ctl::hold), since a pass repeated on its own
// output may overflow -- which does not change what a launch costs.
tbs_status tbs_profile_term(tbs_plan *pl, int ifreq, int reps, double out_ms[4], void *stream) {
    if (pl) ++pl->epoch;
    if (!pl || !out_ms || reps < 1 || reps > 256 || ifreq < 0 || ifreq >= (int)pl->fr.size()) return TBS_ERR_INVALID_ARG;
    tbs_status ws = ensure_workspace(pl);
    if (ws != TBS_OK) return ws;
    Freq &f = pl->fr[ifreq];
    Slot &s = pl->slot[0];
    if (!f.have_V || !f.have_S) return fail(pl, TBS_ERR_NOT_READY, "medium and source required");
    cudaStream_t st = (cudaStream_t)stream;
    tbs_status hs = ensure_history(pl, (reps + 1) * 2 + 8);
    if (hs != TBS_OK) return hs;
    Ctl *h = s.h_ctl;
    memset(&h[0], 0, sizeof(Ctl));
    h[0].max_terms = 1 << 30;
    h[0].tol = 0.0;
    h[0].hold = 1;
    CU(pl, cudaMemcpyAsync(f.ctl, &h[0], sizeof(Ctl), cudaMemcpyHostToDevice, st));
    CU(pl, cudaMemsetAsync(s.norms, 0, sizeof(double) * 2 * pl->hist_cap, st));
    RowArgs r;
    fill_row_args(pl, f, s, r, f.S, (float)(1.0 / (f.k0 * f.k0)), 1);
    CU(pl, launch_row(pl->n[0], true, r, st));
    for (int i = 0; i < 3; ++i) CU(pl, launch_term(pl, f, s, st));
    const int nmid = mid_launches(pl);
    fill_row_args(pl, f, s, r, nullptr, 0.f, 1);
    for (int k = 0; k < 4; ++k) out_ms[k] = 0.0;
    tbs_status res = TBS_OK;
    LaunchOpt popt;
    popt.overlap = pl->overlap != 0;
    // out_ms[0] = row kernel, out_ms[1..] = column/plane passes in launch order
    for (int k = 0; k <= nmid && res == TBS_OK; ++k) {
        cudaError_t e = cudaEventRecord(pl->ev_b0, st);
        for (int i = 0; i < reps && e == cudaSuccess; ++i)
            e = k < nmid ? launch_mid_passes(pl, f, s, st, k, popt) : launch_row(pl->n[0], false, r, st, false, popt);
        if (e == cudaSuccess) e = cudaEventRecord(pl->ev_b1, st);
        if (e == cudaSuccess) e = cudaStreamSynchronize(st);
        float ms = 0.f;
        if (e == cudaSuccess) e = cudaEventElapsedTime(&ms, pl->ev_b0, pl->ev_b1);
        if (e != cudaSuccess) res = fail(pl, TBS_ERR_CUDA, "tbs_profile_term: %s", cudaGetErrorString(e));
        out_ms[k == nmid ? 0 : k + 1] = ms / reps;
    }
    return res;
}

}  // extern "C"
