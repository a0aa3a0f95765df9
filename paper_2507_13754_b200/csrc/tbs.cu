// tbs.cu -- C ABI of libtbs (include/tbs.h): plan management, setup and the Born-term loop.
// No CPU fallback: every compute entry point needs a CUDA device.
#include "../../include/tbs.h"

#include <cmath>
#include <cstdarg>
#include <cstdio>
#include <cstring>
#include <string>
#include <vector>

#include "dispatch.cuh"
#include "setup_kernels.cuh"

using namespace tbs;

namespace {

constexpr double kPi = 3.14159265358979323846;
constexpr int kMaxSlots = 4;          // members of a frequency batch in flight at once, at most
constexpr size_t kWsAlign = 256;      // alignment of every workspace region (TMA / bulk copies need 16)

// A CUDA graph of `batch` Born terms of one frequency on one slot at one grid width.
struct TermGraph {
    cudaGraphExec_t exec = nullptr;
    int batch = 0;
};

struct Freq {
    double f = 0, omega = 0, k0 = 0;
    float2 *V = nullptr;      // [n] V/k0^2                     (workspace)
    float2 *S = nullptr;      // [n] source density             (workspace)
    float2 *p = nullptr;      // [n] running field              (workspace)
    float2 *ucbs = nullptr;   // [n] current term of the convergent Born series (allocated by tbs_set_scheme)
    float *p2[3] = {nullptr, nullptr, nullptr};  // per-axis |p|^2/k0^2, position order, [2 n[a]]
    Ctl *ctl = nullptr;
    TermGraph graph[kMaxSlots][2];   // [slot][0 = all SMs, 1 = half of them]
    bool have_V = false, have_S = false;
    KAbs kabs = {0.f, 0.f, 0.f, 0.f};  // nu > 0: k-space multiplier potential of Eq. 24 instead of V(r)
};

// What one series in flight needs beyond its frequency's V, S, p: the transform intermediates, the norm and
// history buffers, the host mirrors and the events of the batched loop.  Slot 0 serves every single solve;
// slot 1 exists for plans with more than one frequency (two members of the batch are in flight at once).
struct Slot {
    float2 *W1 = nullptr;   // [nz*ny][2 nx]                    (workspace)
    float2 *W2 = nullptr;   // 3-D: [nz][2 ny][2 nx]            (workspace)
    bool own_w = false;     // slots beyond the second: W1/W2 allocated by the plan (tbs_set_concurrency)
    CUtensorMap conv_map;   // tensor map of the array k_conv transforms in place (W1 in 2-D, W2 in 3-D)
    double *norms = nullptr, *history = nullptr;   // device, hist_cap entries
    double *h_hist = nullptr;                      // pinned
    Ctl *h_ctl = nullptr;                          // pinned, 4 entries
    cudaStream_t own_stream = nullptr;             // batch members run on the slot's own stream
    cudaEvent_t ev[2] = {nullptr, nullptr}, ev_t0 = nullptr, ev_t1 = nullptr, ev_join = nullptr;
};

}  // namespace

struct tbs_plan {
    int ndim = 2;
    int n[3] = {1, 1, 1};
    long long npts = 0;
    double dx = 0, c0 = 0, damping = 0;
    double beta = 1.0, rho0 = 1000.0;
    std::vector<Freq> fr;
    int nslots = 1;              // slots with streams, events and history buffers: min(nfreq, kMaxSlots)
    int ws_slots = 1;            // slots whose W1/W2 live in the workspace: min(nfreq, 2)
    Slot slot[kMaxSlots];
    float2 *lutA[3] = {nullptr, nullptr, nullptr};   // per axis, fft_engine.cuh "Luts"
    float2 *lutB[3] = {nullptr, nullptr, nullptr};
    float2 *lutC[3] = {nullptr, nullptr, nullptr};
    float4 *lutAB[3] = {nullptr, nullptr, nullptr};
    float *abl[3] = {nullptr, nullptr, nullptr};
    // workspace: V, S, p of every frequency and W1 (W2) of every slot, in one device range that the caller
    // may own (tbs_plan_set_workspace) -- otherwise allocated by the plan at first use
    void *ws = nullptr;
    size_t ws_bytes = 0;
    bool ws_owned = false;
    int hist_cap = 0;
    unsigned int *maxbits = nullptr;
    void *stage = nullptr;       // device staging of tbs_set_source (positions, amplitudes), grows only
    size_t stage_bytes = 0;
    cudaEvent_t ev_fork = nullptr, ev_b0 = nullptr, ev_b1 = nullptr;
    size_t small_bytes = 0;      // device bytes outside the workspace (tables, control)
    int graph_batch = 16;
    int concurrency = 2;         // members in flight (tbs_set_concurrency)
    unsigned long long epoch = 0;         // bumped by every call that changes what a series computes or its state
    unsigned long long resume_epoch = ~0ull;  // epoch at the end of a capped single-frequency solve (tbs_solve_resume)
    int twof = 0;                // tbs_set_kspace_scatterer: the two-field form of the periodic kernels
    int overlap = 0;             // programmatic dependent launch of the term kernels (measured slower: off)
    int scheme = TBS_SCHEME_BORN;
    int boundary = TBS_BOUNDARY_PAD;
    int crit_row = -1;
    long long launches = 0;
    double loop_ms = 0;
    int sms = 0;
    std::string err;
};

namespace {

tbs_status fail(tbs_plan *p, tbs_status st, const char *fmt, ...) {
    if (p) {
        char buf[512];
        va_list ap;
        va_start(ap, fmt);
        vsnprintf(buf, sizeof buf, fmt, ap);
        va_end(ap);
        p->err = buf;
    }
    return st;
}

#define CU(plan, call)                                                                      \
    do {                                                                                    \
        cudaError_t e_ = (call);                                                            \
        if (e_ != cudaSuccess)                                                              \
            return fail(plan, e_ == cudaErrorMemoryAllocation ? TBS_ERR_ALLOC : TBS_ERR_CUDA, \
                        "%s: %s", #call, cudaGetErrorString(e_));                           \
    } while (0)

template <class T>
cudaError_t dmalloc(tbs_plan *p, T **ptr, size_t count) {
    cudaError_t e = cudaMalloc((void **)ptr, count * sizeof(T));
    if (e == cudaSuccess) p->small_bytes += count * sizeof(T);
    return e;
}

bool pow2(int v) { return v > 0 && (v & (v - 1)) == 0; }
inline unsigned nblk(long long n, int b) { return (unsigned)((n + b - 1) / b); }
inline size_t align_up(size_t v) { return (v + kWsAlign - 1) / kWsAlign * kWsAlign; }

// Periodic boundary in 2-D: the unpadded kernels (one N-point transform per line, W1 is [ny][nx]); in 3-D the
// padded kernels with masked axis tables.
bool per_mode(const tbs_plan *pl) { return pl->boundary == TBS_BOUNDARY_PERIODIC && pl->ndim == 2; }
// How the kernels use the two lanes of a packed value: 0 the parity halves of a padded line, 1 two lines of the
// unpadded periodic form, 2 two fields of one line (k-space multiplier plus a scatterer, periodic form).
int lane_mode(const tbs_plan *pl) { return per_mode(pl) ? (pl->twof ? 2 : 1) : 0; }

size_t w1_elems(const tbs_plan *pl) { return (size_t)pl->n[1] * pl->n[2] * 2 * pl->n[0]; }
size_t w2_elems(const tbs_plan *pl) { return pl->ndim == 3 ? (size_t)pl->n[2] * 2 * pl->n[1] * 2 * pl->n[0] : 0; }

// Layout of the workspace: V, S, p of frequency 0, 1, ...; then W1 (and W2) of slot 0, 1.
size_t workspace_layout(tbs_plan *pl, char *base, bool bind) {
    size_t off = 0;
    auto take = [&](size_t elems) {
        float2 *ptr = bind ? reinterpret_cast<float2 *>(base + off) : nullptr;
        off += align_up(elems * sizeof(float2));
        return ptr;
    };
    for (auto &f : pl->fr) {
        float2 *v = take((size_t)pl->npts), *s = take((size_t)pl->npts), *p = take((size_t)pl->npts);
        if (bind) { f.V = v; f.S = s; f.p = p; }
    }
    for (int i = 0; i < pl->ws_slots; ++i) {
        float2 *w1 = take(w1_elems(pl));
        float2 *w2 = pl->ndim == 3 ? take(w2_elems(pl)) : nullptr;
        if (bind) { pl->slot[i].W1 = w1; pl->slot[i].W2 = w2; }
    }
    return off;
}

void destroy_graphs(tbs_plan *pl) {
    for (auto &f : pl->fr)
        for (auto &row : f.graph)
            for (auto &g : row) {
                if (g.exec) cudaGraphExecDestroy(g.exec);
                g.exec = nullptr;
                g.batch = 0;
            }
}

// Tensor maps of the arrays k_conv transforms in place: W1 ([ny][2 nx], or [ny][nx] in the unpadded periodic
// form) in 2-D, W2 in 3-D.
tbs_status make_tensor_maps(tbs_plan *pl) {
    if (!pl->ws) return TBS_OK;
    const long long mx = (lane_mode(pl) == 1 ? 1LL : 2LL) * pl->n[0], my = 2LL * pl->n[1];
    for (int i = 0; i < pl->nslots; ++i) {
        Slot &s = pl->slot[i];
        if (!s.W1) continue;   // a slot beyond the second that tbs_set_concurrency has not asked for
        if (pl->ndim == 2) CU(pl, make_conv_tensor_map(&s.conv_map, s.W1, mx, pl->n[1], mx, conv_tile_width(pl->n[1])));
        else CU(pl, make_conv_tensor_map(&s.conv_map, s.W2, my * mx, pl->n[2], my * mx, conv_tile_width(pl->n[2])));
    }
    return TBS_OK;
}

// Point the plan at a workspace.  Its contents are undefined: medium and source have to be set (again).
tbs_status bind_workspace(tbs_plan *pl, void *base, size_t bytes, bool owned) {
    destroy_graphs(pl);
    if (pl->ws && pl->ws_owned) cudaFree(pl->ws);
    pl->ws = base;
    pl->ws_bytes = bytes;
    pl->ws_owned = owned;
    workspace_layout(pl, (char *)base, true);
    for (auto &f : pl->fr) { f.have_V = false; f.have_S = false; }
    return make_tensor_maps(pl);
}

// Every call that touches V, S, p or W goes through here: without a caller-owned workspace the plan allocates.
tbs_status ensure_workspace(tbs_plan *pl) {
    if (pl->ws) return TBS_OK;
    const size_t bytes = workspace_layout(pl, nullptr, false);
    void *base = nullptr;
    CU(pl, cudaMalloc(&base, bytes));
    return bind_workspace(pl, base, bytes, true);
}

void fill_row_args(tbs_plan *pl, Freq &f, Slot &s, RowArgs &a, const float2 *src, float src_scale, int do_fwd) {
    a.W = s.W1;
    a.src = src;
    a.V = f.V;
    a.p = f.p;
    a.ax = pl->abl[0];
    a.ay = pl->abl[1];
    a.az = pl->ndim == 3 ? pl->abl[2] : nullptr;
    a.ny = pl->n[1];
    a.rows = pl->n[1] * (pl->ndim == 3 ? pl->n[2] : 1);
    a.src_scale = src_scale;
    a.ucbs = pl->scheme == TBS_SCHEME_CBS ? f.ucbs : nullptr;
    a.crit_row = pl->crit_row;
    a.inv_e = (float)(1.0 / pl->damping);
    a.scale = (float)(1.0 / (8.0 * (double)pl->npts) * (pl->ndim == 2 ? 2.0 : 1.0) / pl->damping);
    if (pl->boundary == TBS_BOUNDARY_PERIODIC) a.scale *= (float)(1 << pl->ndim);  // the odd half carries nothing
    a.do_fwd = do_fwd;
    a.per = lane_mode(pl);
    a.norms = s.norms;
    a.history = s.history;
    a.ctl = f.ctl;
    a.lut = Luts{pl->lutA[0], pl->lutB[0], pl->lutC[0], pl->lutAB[0]};
}

// Column / plane passes of one term (K2 in 2-D; y-forward, z-conv, y-inverse in 3-D).
cudaError_t launch_mid_passes(tbs_plan *pl, Freq &f, Slot &s, cudaStream_t st, int which = -1, LaunchOpt opt = LaunchOpt()) {
    const int nx = pl->n[0], ny = pl->n[1], nz = pl->n[2];
    const long long mx = (lane_mode(pl) == 1 ? 1LL : 2LL) * nx, my = 2LL * ny;
    ColArgs a;
    memset(&a, 0, sizeof a);
    a.ctl = f.ctl;
    a.inv_e = (float)(1.0 / pl->damping);
    a.kabs = f.kabs;
    a.per = lane_mode(pl);
    a.masked = pl->boundary == TBS_BOUNDARY_PERIODIC && !a.per;
    a.inner_len = (int)mx;
    cudaError_t e = cudaSuccess;
    if (pl->ndim == 2) {
        a.in = s.W1; a.out = s.W1;
        a.lut = Luts{pl->lutA[1], pl->lutB[1], pl->lutC[1], pl->lutAB[1]};
        a.in_line_stride = a.out_line_stride = mx;
        a.p2_line = (const float2 *)f.p2[1]; a.p2_inner = f.p2[0]; a.p2_outer = nullptr;
        if (which < 0 || which == 0) e = launch_conv(ny, a, &s.conv_map, 1, st, false, opt);
        return e;
    }
    // y forward: W1[z][y][kx] -> W2[z][ky][kx]
    if (which < 0 || which == 0) {
        a.in = s.W1; a.out = s.W2;
        a.lut = Luts{pl->lutA[1], pl->lutB[1], pl->lutC[1], pl->lutAB[1]};
        a.in_line_stride = mx; a.out_line_stride = mx;
        a.in_outer_stride = (long long)ny * mx; a.out_outer_stride = my * mx;
        e = launch_col(ny, MODE_FWD, a, nz, st, false, opt);
        if (e != cudaSuccess) return e;
    }
    // z convolution, in place on W2; lines (ky, kx), outer = ky
    if (which < 0 || which == 1) {
        a.in = s.W2; a.out = s.W2;
        a.lut = Luts{pl->lutA[2], pl->lutB[2], pl->lutC[2], pl->lutAB[2]};
        a.in_line_stride = a.out_line_stride = my * mx;
        a.in_outer_stride = a.out_outer_stride = mx;
        a.p2_line = (const float2 *)f.p2[2]; a.p2_inner = f.p2[0]; a.p2_outer = f.p2[1];
        e = launch_conv(nz, a, &s.conv_map, (int)my, st, false, opt);
        if (e != cudaSuccess) return e;
    }
    // y inverse: W2[z][ky][kx] -> W1[z][y][kx]
    if (which < 0 || which == 2) {
        a.in = s.W2; a.out = s.W1;
        a.lut = Luts{pl->lutA[1], pl->lutB[1], pl->lutC[1], pl->lutAB[1]};
        a.in_line_stride = mx; a.out_line_stride = mx;
        a.in_outer_stride = my * mx; a.out_outer_stride = (long long)ny * mx;
        a.p2_line = nullptr; a.p2_inner = nullptr; a.p2_outer = nullptr;
        e = launch_col(ny, MODE_INV, a, nz, st, false, opt);
    }
    return e;
}

int mid_launches(const tbs_plan *pl) { return pl->ndim == 2 ? 1 : 3; }

cudaError_t launch_term(tbs_plan *pl, Freq &f, Slot &s, cudaStream_t st, LaunchOpt opt = LaunchOpt()) {
    cudaError_t e = launch_mid_passes(pl, f, s, st, -1, opt);
    if (e != cudaSuccess) return e;
    RowArgs r;
    fill_row_args(pl, f, s, r, nullptr, 0.f, 1);
    return launch_row(pl->n[0], false, r, st, false, opt);
}

// Green's-spectrum axis tables of one frequency, in the order each kernel reads them (setup_kernels.cuh).
cudaError_t fill_axis_tables(tbs_plan *pl, Freq &f) {
    for (int a = 0; a < pl->ndim; ++a) {
        int r1, r2, rl;
        radices_of(pl->n[a], r1, r2, rl);
        k_axis_table<<<nblk(2 * pl->n[a], 256), 256>>>(f.p2[a], pl->n[a], r1, r2, rl, pl->dx, f.k0,
                                                        a == 0 || a == pl->ndim - 1,
                                                        a == pl->ndim - 1 ? 1.0 / pl->damping : 1.0,
                                                        per_mode(pl) ? 2 : pl->boundary == TBS_BOUNDARY_PERIODIC);
    }
    return cudaGetLastError();
}

cudaError_t set_kernel_attrs(tbs_plan *pl) {
    ColArgs ca; memset(&ca, 0, sizeof ca);
    RowArgs ra; memset(&ra, 0, sizeof ra);
    cudaError_t e;
    if ((e = launch_row(pl->n[0], true, ra, 0, true)) != cudaSuccess) return e;
    if (pl->ndim == 2) return launch_conv(pl->n[1], ca, nullptr, 1, 0, true);
    if ((e = launch_col(pl->n[1], MODE_FWD, ca, 1, 0, true)) != cudaSuccess) return e;
    return launch_conv(pl->n[2], ca, nullptr, 1, 0, true);
}

// Norm and history buffers of every slot for series of up to max_terms terms.  The captured graphs hold these
// pointers, so a reallocation drops the graphs.
tbs_status ensure_history(tbs_plan *pl, int max_terms, bool keep = false) {
    if (max_terms + 1 <= pl->hist_cap) return TBS_OK;
    destroy_graphs(pl);
    const int cap = max_terms + 1, old_cap = pl->hist_cap;
    for (int i = 0; i < pl->nslots; ++i) {
        Slot &s = pl->slot[i];
        double *norms = nullptr, *history = nullptr, *h_hist = nullptr;
        CU(pl, cudaMalloc((void **)&norms, sizeof(double) * 2 * cap));
        CU(pl, cudaMalloc((void **)&history, sizeof(double) * cap));
        CU(pl, cudaMallocHost((void **)&h_hist, sizeof(double) * cap));
        CU(pl, cudaMemset(norms, 0, sizeof(double) * 2 * cap));
        CU(pl, cudaMemset(history, 0, sizeof(double) * cap));
        if (keep && s.norms && old_cap > 0) {   // tbs_solve_resume: the series so far stays
            CU(pl, cudaMemcpy(norms, s.norms, sizeof(double) * 2 * old_cap, cudaMemcpyDeviceToDevice));
            CU(pl, cudaMemcpy(history, s.history, sizeof(double) * old_cap, cudaMemcpyDeviceToDevice));
        }
        if (s.norms) cudaFree(s.norms);
        if (s.history) cudaFree(s.history);
        if (s.h_hist) cudaFreeHost(s.h_hist);
        s.norms = norms; s.history = history; s.h_hist = h_hist;
    }
    pl->hist_cap = cap;
    return TBS_OK;
}

// Grow-only device staging buffer (tbs_set_source).
tbs_status ensure_stage(tbs_plan *pl, size_t bytes) {
    if (bytes <= pl->stage_bytes) return TBS_OK;
    if (pl->stage) cudaFree(pl->stage);
    pl->stage = nullptr;
    pl->stage_bytes = 0;
    const size_t cap = bytes < 65536 ? 65536 : bytes * 2;
    CU(pl, cudaMalloc(&pl->stage, cap));
    pl->stage_bytes = cap;
    return TBS_OK;
}

}  // namespace

extern "C" {

const char *tbs_version(void) { return "tbs-b200 0.2 (sm_100a)"; }

const char *tbs_last_error(const tbs_plan *plan) { return plan ? plan->err.c_str() : "null plan"; }

size_t tbs_plan_workspace_bytes(const tbs_plan *plan) {
    return plan ? workspace_layout(const_cast<tbs_plan *>(plan), nullptr, false) : 0;
}

tbs_status tbs_plan_set_workspace(tbs_plan *pl, void *dev_ptr, size_t bytes) {
    if (pl) ++pl->epoch;
    if (!pl || !dev_ptr) return TBS_ERR_INVALID_ARG;
    if (((uintptr_t)dev_ptr % kWsAlign) != 0) return fail(pl, TBS_ERR_INVALID_ARG, "workspace must be 256-byte aligned");
    const size_t need = workspace_layout(pl, nullptr, false);
    if (bytes < need) return fail(pl, TBS_ERR_INVALID_ARG, "workspace of %zu bytes, %zu needed", bytes, need);
    cudaPointerAttributes at;
    if (cudaPointerGetAttributes(&at, dev_ptr) != cudaSuccess || at.type != cudaMemoryTypeDevice) {
        cudaGetLastError();
        return fail(pl, TBS_ERR_INVALID_ARG, "workspace is not device memory");
    }
    CU(pl, cudaDeviceSynchronize());
    return bind_workspace(pl, dev_ptr, bytes, false);
}

size_t tbs_plan_device_bytes(const tbs_plan *plan) {
    return plan ? plan->small_bytes + (plan->ws_owned ? plan->ws_bytes : 0) : 0;
}

double tbs_grid_harmonic_frequency(int m, double c0, int n, double dx_m) {
    return (m > 0 && n > 0 && dx_m > 0 && c0 > 0) ? (double)m * c0 / ((double)n * dx_m) : 0.0;
}

int64_t tbs_last_launch_count(const tbs_plan *plan) { return plan ? plan->launches : 0; }
double tbs_last_loop_ms(const tbs_plan *plan) { return plan ? plan->loop_ms : 0.0; }

tbs_status tbs_set_graph_batch(tbs_plan *plan, int terms_per_graph) {
    if (!plan || terms_per_graph < 0 || terms_per_graph > 1024) return TBS_ERR_INVALID_ARG;
    plan->graph_batch = terms_per_graph;
    destroy_graphs(plan);
    return TBS_OK;
}

tbs_status tbs_set_launch_overlap(tbs_plan *plan, int on) {
    if (!plan) return TBS_ERR_INVALID_ARG;
    plan->overlap = on ? 1 : 0;
    destroy_graphs(plan);
    return TBS_OK;
}

tbs_status tbs_set_concurrency(tbs_plan *plan, int members) {
    if (!plan || members < 1 || members > kMaxSlots) return TBS_ERR_INVALID_ARG;
    tbs_plan *pl = plan;
    // the first two slots' intermediates are part of the workspace; further ones are the plan's own
    bool grew = false;
    for (int i = pl->ws_slots; i < members && i < pl->nslots; ++i) {
        Slot &s = pl->slot[i];
        if (s.W1) continue;
        CU(pl, dmalloc(pl, &s.W1, w1_elems(pl)));
        if (pl->ndim == 3) CU(pl, dmalloc(pl, &s.W2, w2_elems(pl)));
        s.own_w = true;
        grew = true;
    }
    if (grew) {
        tbs_status ms = make_tensor_maps(pl);
        if (ms != TBS_OK) return ms;
    }
    plan->concurrency = members;
    return TBS_OK;
}

void tbs_plan_destroy(tbs_plan *pl) {
    if (!pl) return;
    cudaDeviceSynchronize();
    destroy_graphs(pl);
    for (auto &f : pl->fr) {
        cudaFree(f.ctl); cudaFree(f.ucbs);
        for (int a = 0; a < 3; ++a) cudaFree(f.p2[a]);
    }
    if (pl->ws && pl->ws_owned) cudaFree(pl->ws);
    for (int a = 0; a < 3; ++a) { cudaFree(pl->lutA[a]); cudaFree(pl->lutB[a]); cudaFree(pl->lutC[a]); cudaFree(pl->lutAB[a]); }
    for (int a = 0; a < 3; ++a) cudaFree(pl->abl[a]);
    cudaFree(pl->maxbits);
    cudaFree(pl->stage);
    for (auto &s : pl->slot) {
        if (s.own_w) { cudaFree(s.W1); cudaFree(s.W2); }
        cudaFree(s.norms); cudaFree(s.history);
        if (s.h_ctl) cudaFreeHost(s.h_ctl);
        if (s.h_hist) cudaFreeHost(s.h_hist);
        for (int i = 0; i < 2; ++i) if (s.ev[i]) cudaEventDestroy(s.ev[i]);
        if (s.ev_t0) cudaEventDestroy(s.ev_t0);
        if (s.ev_t1) cudaEventDestroy(s.ev_t1);
        if (s.ev_join) cudaEventDestroy(s.ev_join);
        if (s.own_stream) cudaStreamDestroy(s.own_stream);
    }
    if (pl->ev_fork) cudaEventDestroy(pl->ev_fork);
    if (pl->ev_b0) cudaEventDestroy(pl->ev_b0);
    if (pl->ev_b1) cudaEventDestroy(pl->ev_b1);
    delete pl;
}

tbs_status tbs_plan_create(tbs_plan **out, int ndim, const int32_t n[3], double dx_m, int nfreq,
                           const double *f_hz, double c0, double damping) {
    if (!out) return TBS_ERR_INVALID_ARG;
    *out = nullptr;
    if ((ndim != 2 && ndim != 3) || !n || !f_hz || nfreq < 1 || !(dx_m > 0) || !(c0 > 0) || !(damping > 0))
        return TBS_ERR_INVALID_ARG;
    const int nmax = ndim == 2 ? 4096 : 512;
    for (int a = 0; a < ndim; ++a)
        if (!pow2(n[a]) || n[a] < 32 || n[a] > nmax) return TBS_ERR_UNSUPPORTED_SIZE;
    for (int i = 0; i < nfreq; ++i)
        if (!(f_hz[i] > 0)) return TBS_ERR_INVALID_ARG;
    int ndev = 0;
    if (cudaGetDeviceCount(&ndev) != cudaSuccess || ndev == 0) return TBS_ERR_CUDA;

    tbs_plan *pl = new tbs_plan();
    pl->ndim = ndim;
    for (int a = 0; a < ndim; ++a) pl->n[a] = n[a];
    pl->npts = (long long)pl->n[0] * pl->n[1] * pl->n[2];
    pl->dx = dx_m; pl->c0 = c0; pl->damping = damping;
    pl->fr.resize(nfreq);
    pl->nslots = nfreq < kMaxSlots ? nfreq : kMaxSlots;
    pl->ws_slots = nfreq < 2 ? nfreq : 2;
    tbs_status st = TBS_OK;
    auto build = [&]() -> tbs_status {
        int dev = 0;
        CU(pl, cudaGetDevice(&dev));
        CU(pl, cudaDeviceGetAttribute(&pl->sms, cudaDevAttrMultiProcessorCount, dev));
        CU(pl, set_kernel_attrs(pl));
        for (int a = 0; a < ndim; ++a) {
            int r1, r2, rl;
            radices_of(pl->n[a], r1, r2, rl);
            const int N = pl->n[a];
            CU(pl, dmalloc(pl, &pl->lutA[a], N));
            CU(pl, dmalloc(pl, &pl->lutB[a], N));
            k_stage_lut<<<nblk(N, 256), 256>>>(pl->lutA[a], N, r1, 0);
            k_stage_lut<<<nblk(N, 256), 256>>>(pl->lutB[a], N, r1, 1);
            CU(pl, dmalloc(pl, &pl->lutAB[a], N));
            k_stage_lut_ab<<<nblk(N, 256), 256>>>(pl->lutAB[a], N, r1, 0);
            if (r2 > 0) {
                CU(pl, dmalloc(pl, &pl->lutC[a], N / r1));
                k_stage_lut<<<nblk(N / r1, 256), 256>>>(pl->lutC[a], N / r1, r2, 0);
            }
            CU(pl, cudaGetLastError());
        }
        for (int a = 0; a < ndim; ++a) {
            CU(pl, dmalloc(pl, &pl->abl[a], pl->n[a]));
            k_abl_window<<<nblk(pl->n[a], 256), 256>>>(pl->abl[a], pl->n[a], 0, 0.0);
        }
        CU(pl, cudaGetLastError());
        CU(pl, dmalloc(pl, &pl->maxbits, 1));
        for (int i = 0; i < pl->nslots; ++i) {
            Slot &s = pl->slot[i];
            CU(pl, cudaMallocHost((void **)&s.h_ctl, sizeof(Ctl) * 4));
            for (int k = 0; k < 2; ++k) CU(pl, cudaEventCreateWithFlags(&s.ev[k], cudaEventDisableTiming));
            CU(pl, cudaEventCreate(&s.ev_t0));
            CU(pl, cudaEventCreate(&s.ev_t1));
            CU(pl, cudaEventCreateWithFlags(&s.ev_join, cudaEventDisableTiming));
            if (pl->nslots > 1) CU(pl, cudaStreamCreateWithFlags(&s.own_stream, cudaStreamNonBlocking));
        }
        CU(pl, cudaEventCreateWithFlags(&pl->ev_fork, cudaEventDisableTiming));
        CU(pl, cudaEventCreate(&pl->ev_b0));
        CU(pl, cudaEventCreate(&pl->ev_b1));
        for (int i = 0; i < nfreq; ++i) {
            Freq &f = pl->fr[i];
            f.f = f_hz[i];
            f.omega = 2.0 * kPi * f.f;
            f.k0 = f.omega / c0;
            CU(pl, dmalloc(pl, &f.ctl, 1));
            for (int a = 0; a < ndim; ++a) CU(pl, dmalloc(pl, &f.p2[a], 2 * pl->n[a]));
            CU(pl, fill_axis_tables(pl, f));
        }
        CU(pl, cudaDeviceSynchronize());
        return TBS_OK;
    };
    st = build();
    if (st != TBS_OK) {
        // keep the message reachable through a failed create: print it
        fprintf(stderr, "tbs_plan_create: %s\n", pl->err.c_str());
        tbs_plan_destroy(pl);
        return st;
    }
    *out = pl;
    return TBS_OK;
}

__global__ void k_fill_complex(float2 *dst, float2 v, long long n) {
    const long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (i < n) dst[i] = v;
}

tbs_status tbs_set_kspace_absorption(tbs_plan *pl, double alpha0_si, double nu, int dispersive) {
    if (pl) ++pl->epoch;
    if (!pl || !(alpha0_si >= 0.0)) return TBS_ERR_INVALID_ARG;
    if (alpha0_si > 0.0 && (!(nu > 0.0) || nu > 2.0 || fabs(nu - 1.0) < 1e-9))
        return fail(pl, TBS_ERR_INVALID_ARG, "power-law exponent must lie in (0, 2] and differ from 1 (PAPER.md:53)");
    if (alpha0_si > 0.0 && pl->scheme == TBS_SCHEME_CBS)
        return fail(pl, TBS_ERR_INVALID_ARG, "the k-space multiplier potential is not combined with TBS_SCHEME_CBS");
    tbs_status ws = ensure_workspace(pl);
    if (ws != TBS_OK) return ws;
    CU(pl, cudaDeviceSynchronize());
    if (pl->twof) {
        pl->twof = 0;   // back to the multiplier alone (or to the spatial potential): W is one field wide again
        tbs_status ms = make_tensor_maps(pl);
        if (ms != TBS_OK) return ms;
    }
    for (auto &f : pl->fr) {
        if (alpha0_si == 0.0) {
            if (f.kabs.nu > 0.f) f.have_V = false;  // the spatial potential has to be set again
            f.kabs = KAbs{0.f, 0.f, 0.f, 0.f};
            continue;
        }
        // tau = -2 alpha0 v_f^(nu-1), eta = 2 alpha0 v_f^nu tan(pi nu/2)
        const double tau = -2.0 * alpha0_si * pow(pl->c0, nu - 1.0);
        const double eta = dispersive ? 2.0 * alpha0_si * pow(pl->c0, nu) * tan(kPi * nu / 2.0) : 0.0;
        f.kabs.A = (float)(tau * f.omega * pow(f.k0, nu - 2.0));
        f.kabs.B = (float)(eta * pow(f.k0, nu - 1.0));
        f.kabs.nu = (float)nu;
        f.kabs.e = (float)pl->damping;
        k_fill_complex<<<nblk(pl->npts, 256), 256>>>(f.V, make_float2(1.f, 0.f), pl->npts);  // the term passes unmultiplied
        f.have_V = true;
    }
    destroy_graphs(pl);
    CU(pl, cudaGetLastError());
    CU(pl, cudaDeviceSynchronize());
    return TBS_OK;
}

tbs_status tbs_set_boundary(tbs_plan *pl, int boundary) {
    if (pl) ++pl->epoch;
    if (!pl || (boundary != TBS_BOUNDARY_PAD && boundary != TBS_BOUNDARY_PERIODIC)) return TBS_ERR_INVALID_ARG;
    CU(pl, cudaDeviceSynchronize());
    pl->boundary = boundary;
    if (pl->twof && !per_mode(pl)) {   // the two-field form exists on the periodic kernels only
        pl->twof = 0;
        for (auto &f : pl->fr) f.have_V = false;
    }
    for (auto &f : pl->fr) CU(pl, fill_axis_tables(pl, f));
    // first/last-stage twiddles: the odd lane carries the padding twist, or (unpadded periodic form) a second line
    for (int a = 0; a < pl->ndim; ++a) {
        int r1, r2, rl;
        radices_of(pl->n[a], r1, r2, rl);
        k_stage_lut_ab<<<nblk(pl->n[a], 256), 256>>>(pl->lutAB[a], pl->n[a], r1, per_mode(pl) ? 1 : 0);
    }
    CU(pl, cudaGetLastError());
    tbs_status ms = make_tensor_maps(pl);
    if (ms != TBS_OK) return ms;
    destroy_graphs(pl);  // the captured launches carry the normalisation
    CU(pl, cudaDeviceSynchronize());
    return TBS_OK;
}

tbs_status tbs_set_criterion(tbs_plan *pl, int criterion, int row) {
    if (pl) ++pl->epoch;
    if (!pl || (criterion != TBS_CRIT_L2_GRID && criterion != TBS_CRIT_L1_ROW)) return TBS_ERR_INVALID_ARG;
    const int rows = pl->n[1] * (pl->ndim == 3 ? pl->n[2] : 1);
    if (criterion == TBS_CRIT_L1_ROW && (row < 0 || row >= rows)) return fail(pl, TBS_ERR_INVALID_ARG, "row outside the grid");
    pl->crit_row = criterion == TBS_CRIT_L1_ROW ? row : -1;
    destroy_graphs(pl);
    return TBS_OK;
}

tbs_status tbs_set_scheme(tbs_plan *pl, int scheme) {
    if (pl) ++pl->epoch;
    if (!pl || (scheme != TBS_SCHEME_BORN && scheme != TBS_SCHEME_CBS)) return TBS_ERR_INVALID_ARG;
    if (scheme == TBS_SCHEME_CBS) {
        for (auto &f : pl->fr)
            if (f.kabs.nu > 0.f)
                return fail(pl, TBS_ERR_INVALID_ARG, "TBS_SCHEME_CBS is not combined with the k-space multiplier potential");
        for (auto &f : pl->fr)
            if (!f.ucbs) CU(pl, dmalloc(pl, &f.ucbs, (size_t)pl->npts));
    }
    if (scheme != pl->scheme) destroy_graphs(pl);  // the captured launches carry the scheme
    pl->scheme = scheme;
    return TBS_OK;
}

tbs_status tbs_set_abl(tbs_plan *pl, int cells, double zeta_half_mu) {
    if (pl) ++pl->epoch;
    if (!pl || cells < 0) return TBS_ERR_INVALID_ARG;
    for (int a = 0; a < pl->ndim; ++a)
        if (2 * cells > pl->n[a]) return fail(pl, TBS_ERR_INVALID_ARG, "ABL wider than half the grid");
    for (int a = 0; a < pl->ndim; ++a)
        k_abl_window<<<nblk(pl->n[a], 256), 256>>>(pl->abl[a], pl->n[a], cells, zeta_half_mu);
    CU(pl, cudaGetLastError());
    CU(pl, cudaDeviceSynchronize());
    return TBS_OK;
}

// A spatial potential replaces the k-space multiplier of Eq. 24, if one was active (the two are not combined).
static void drop_kspace_potential(tbs_plan *pl, Freq &f) {
    if (f.kabs.nu > 0.f) {
        f.kabs = KAbs{0.f, 0.f, 0.f, 0.f};
        destroy_graphs(pl);
    }
    if (pl->twof) {
        cudaDeviceSynchronize();
        pl->twof = 0;
        make_tensor_maps(pl);
        destroy_graphs(pl);
    }
}

tbs_status tbs_set_kspace_scatterer(tbs_plan *pl, const float *c, void *stream) {
    if (pl) ++pl->epoch;
    if (!pl || !c) return TBS_ERR_INVALID_ARG;
    if (!per_mode(pl))
        return fail(pl, TBS_ERR_INVALID_ARG, "the multiplier plus a scatterer runs on the periodic boundary in 2-D (the paper's form)");
    for (auto &f : pl->fr)
        if (!(f.kabs.nu > 0.f)) return fail(pl, TBS_ERR_NOT_READY, "tbs_set_kspace_absorption first");
    if (pl->scheme == TBS_SCHEME_CBS) return fail(pl, TBS_ERR_INVALID_ARG, "not combined with TBS_SCHEME_CBS");
    tbs_status ws = ensure_workspace(pl);
    if (ws != TBS_OK) return ws;
    cudaStream_t st = (cudaStream_t)stream;
    CU(pl, cudaDeviceSynchronize());
    for (auto &f : pl->fr) {
        k_scatterer_potential<<<nblk(pl->npts, 256), 256, 0, st>>>(f.V, c, f.omega, f.k0, pl->npts);
        f.have_V = true;
    }
    CU(pl, cudaGetLastError());
    CU(pl, cudaStreamSynchronize(st));
    if (!pl->twof) {
        pl->twof = 1;
        tbs_status ms = make_tensor_maps(pl);
        if (ms != TBS_OK) return ms;
    }
    destroy_graphs(pl);
    return TBS_OK;
}

tbs_status tbs_set_medium(tbs_plan *pl, const float *c, const float *rho, const float *alpha0_map,
                          double alpha0_db, double y, double beta, double rho0, void *stream) {
    if (pl) ++pl->epoch;
    if (!pl || !c) return TBS_ERR_INVALID_ARG;
    const bool absorbing = alpha0_map != nullptr || alpha0_db != 0.0;
    if (absorbing && fabs(y - 1.0) < 1e-9) return fail(pl, TBS_ERR_INVALID_ARG, "y = 1 is excluded (PAPER.md:53)");
    if (!(rho0 > 0)) return fail(pl, TBS_ERR_INVALID_ARG, "rho0 must be positive");
    (void)rho;  // density does not enter V; rho0 feeds xi of the harmonic source
    tbs_status ws = ensure_workspace(pl);
    if (ws != TBS_OK) return ws;
    cudaStream_t st = (cudaStream_t)stream;
    pl->beta = beta;
    pl->rho0 = rho0;
    for (auto &f : pl->fr) {
        drop_kspace_potential(pl, f);
        k_potential<<<nblk(pl->npts, 256), 256, 0, st>>>(f.V, c, alpha0_map, alpha0_db, y, f.omega, f.k0,
                                                           pl->damping, pl->npts);
        f.have_V = true;
    }
    CU(pl, cudaGetLastError());
    CU(pl, cudaStreamSynchronize(st));
    return TBS_OK;
}

tbs_status tbs_set_medium_host(tbs_plan *pl, const float *c, const float *rho, const float *alpha0_map,
                               double alpha0_db, double y, double beta, double rho0, void *stream) {
    if (!pl || !c) return TBS_ERR_INVALID_ARG;
    tbs_status ws = ensure_workspace(pl);
    if (ws != TBS_OK) return ws;
    cudaStream_t st = (cudaStream_t)stream;
    // stage through W1 of slot 0 (>= 2 n complex = 4 n floats): c at [0, n), alpha0 map at [n, 2n)
    float *dc = (float *)pl->slot[0].W1;
    float *da = alpha0_map ? dc + pl->npts : nullptr;
    CU(pl, cudaMemcpyAsync(dc, c, sizeof(float) * pl->npts, cudaMemcpyHostToDevice, st));
    if (alpha0_map) CU(pl, cudaMemcpyAsync(da, alpha0_map, sizeof(float) * pl->npts, cudaMemcpyHostToDevice, st));
    (void)rho;  // accepted for symmetry with tbs_set_medium, where it is not read either
    return tbs_set_medium(pl, dc, nullptr, da, alpha0_db, y, beta, rho0, stream);
}

tbs_status tbs_set_potential(tbs_plan *pl, int ifreq, const float *V, void *stream) {
    if (pl) ++pl->epoch;
    if (!pl || !V || ifreq < 0 || ifreq >= (int)pl->fr.size()) return TBS_ERR_INVALID_ARG;
    tbs_status ws = ensure_workspace(pl);
    if (ws != TBS_OK) return ws;
    cudaStream_t st = (cudaStream_t)stream;
    Freq &f = pl->fr[ifreq];
    drop_kspace_potential(pl, f);
    k_scale_complex<<<nblk(pl->npts, 256), 256, 0, st>>>(f.V, (const float2 *)V, 1.0 / (f.k0 * f.k0), pl->npts);
    CU(pl, cudaGetLastError());
    CU(pl, cudaStreamSynchronize(st));
    f.have_V = true;
    return TBS_OK;
}

tbs_status tbs_set_source(tbs_plan *pl, int n_src, const double *pos_m, const float *amp, void *stream) {
    if (pl) ++pl->epoch;
    if (!pl || n_src < 1 || !pos_m || !amp) return TBS_ERR_INVALID_ARG;
    for (int j = 0; j < n_src; ++j)
        for (int a = 0; a < pl->ndim; ++a) {
            const double g = pos_m[(size_t)j * pl->ndim + a] / pl->dx;
            if (!(g >= 0.0) || g > (double)(pl->n[a] - 1))
                return fail(pl, TBS_ERR_INVALID_ARG, "source %d lies outside the grid", j);
        }
    tbs_status ws = ensure_workspace(pl);
    if (ws != TBS_OK) return ws;
    cudaStream_t st = (cudaStream_t)stream;
    const size_t nf = pl->fr.size();
    const size_t pos_bytes = align_up(sizeof(double) * n_src * pl->ndim);
    const size_t amp_bytes = sizeof(float2) * n_src * nf;
    tbs_status ss = ensure_stage(pl, pos_bytes + amp_bytes);
    if (ss != TBS_OK) return ss;
    double *dpos = (double *)pl->stage;
    float2 *damp = (float2 *)((char *)pl->stage + pos_bytes);
    CU(pl, cudaMemcpyAsync(dpos, pos_m, sizeof(double) * n_src * pl->ndim, cudaMemcpyHostToDevice, st));
    CU(pl, cudaMemcpyAsync(damp, amp, amp_bytes, cudaMemcpyHostToDevice, st));
    for (size_t i = 0; i < nf; ++i) {
        Freq &f = pl->fr[i];
        CU(pl, cudaMemsetAsync(f.S, 0, sizeof(float2) * pl->npts, st));
        k_deposit<<<nblk((long long)n_src << pl->ndim, 128), 128, 0, st>>>(f.S, dpos, damp + i * n_src, n_src,
                                                                            pl->ndim, pl->n[0], pl->n[1], pl->n[2], pl->dx);
        f.have_S = true;
    }
    CU(pl, cudaGetLastError());
    CU(pl, cudaStreamSynchronize(st));   // the host arrays may be reused by the caller; the staging by the next call
    return TBS_OK;
}

tbs_status tbs_set_source_field(tbs_plan *pl, int ifreq, const float *S, void *stream) {
    if (pl) ++pl->epoch;
    if (!pl || !S || ifreq < 0 || ifreq >= (int)pl->fr.size()) return TBS_ERR_INVALID_ARG;
    tbs_status ws = ensure_workspace(pl);
    if (ws != TBS_OK) return ws;
    cudaStream_t st = (cudaStream_t)stream;
    Freq &f = pl->fr[ifreq];
    CU(pl, cudaMemcpyAsync(f.S, S, sizeof(float2) * pl->npts, cudaMemcpyDeviceToDevice, st));
    CU(pl, cudaStreamSynchronize(st));
    f.have_S = true;
    return TBS_OK;
}

tbs_status tbs_get_potential(tbs_plan *pl, int ifreq, float *out, void *stream) {
    if (!pl || !out || ifreq < 0 || ifreq >= (int)pl->fr.size()) return TBS_ERR_INVALID_ARG;
    Freq &f = pl->fr[ifreq];
    if (!f.have_V) return fail(pl, TBS_ERR_NOT_READY, "medium not set");
    cudaStream_t st = (cudaStream_t)stream;
    k_scale_complex<<<nblk(pl->npts, 256), 256, 0, st>>>((float2 *)out, f.V, f.k0 * f.k0, pl->npts);
    CU(pl, cudaGetLastError());
    CU(pl, cudaStreamSynchronize(st));
    return TBS_OK;
}

tbs_status tbs_get_source(tbs_plan *pl, int ifreq, float *out, void *stream) {
    if (!pl || !out || ifreq < 0 || ifreq >= (int)pl->fr.size()) return TBS_ERR_INVALID_ARG;
    Freq &f = pl->fr[ifreq];
    if (!f.have_S) return fail(pl, TBS_ERR_NOT_READY, "source not set");
    cudaStream_t st = (cudaStream_t)stream;
    CU(pl, cudaMemcpyAsync(out, f.S, sizeof(float2) * pl->npts, cudaMemcpyDeviceToDevice, st));
    CU(pl, cudaStreamSynchronize(st));
    return TBS_OK;
}

tbs_status tbs_green_spectrum(tbs_plan *pl, int ifreq, float *out, void *stream) {
    if (!pl || !out || ifreq < 0 || ifreq >= (int)pl->fr.size()) return TBS_ERR_INVALID_ARG;
    Freq &f = pl->fr[ifreq];
    cudaStream_t st = (cudaStream_t)stream;
    const int mx = 2 * pl->n[0], my = 2 * pl->n[1], mz = pl->ndim == 3 ? 2 * pl->n[2] : 1;
    const long long tot = (long long)mx * my * mz;
    k_green_spectrum<<<nblk(tot, 256), 256, 0, st>>>((float2 *)out, mx, my, mz, pl->dx, f.k0,
                                                       pl->damping * f.k0 * f.k0);
    CU(pl, cudaGetLastError());
    CU(pl, cudaStreamSynchronize(st));
    return TBS_OK;
}

}  // extern "C"

#include "solve.inl"
