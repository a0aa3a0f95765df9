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

struct Freq {
    double f = 0, omega = 0, k0 = 0;
    float2 *V = nullptr;      // [n] V/k0^2
    float2 *S = nullptr;      // [n] source density
    float2 *p = nullptr;      // [n] running field
    float2 *ucbs = nullptr;   // [n] current term of the convergent Born series (allocated by tbs_set_scheme)
    float *p2[3] = {nullptr, nullptr, nullptr};  // per-axis |p|^2/k0^2, position order, [2 n[a]]
    Ctl *ctl = nullptr;
    cudaGraphExec_t graph = nullptr;
    int graph_batch = 0;
    bool have_V = false, have_S = false;
    KAbs kabs = {0.f, 0.f, 0.f, 0.f};  // nu > 0: k-space multiplier potential of Eq. 24 instead of V(r)
};

}  // namespace

struct tbs_plan {
    int ndim = 2;
    int n[3] = {1, 1, 1};
    long long npts = 0;
    double dx = 0, c0 = 0, damping = 0;
    double beta = 1.0, rho0 = 1000.0;
    std::vector<Freq> fr;
    float2 *lutA[3] = {nullptr, nullptr, nullptr};   // per axis, fft_engine.cuh "Luts"
    float2 *lutB[3] = {nullptr, nullptr, nullptr};
    float2 *lutC[3] = {nullptr, nullptr, nullptr};
    float4 *lutAB[3] = {nullptr, nullptr, nullptr};
    float2 *W1 = nullptr;   // [nz*ny][2 nx]
    float2 *W2 = nullptr;   // 3-D: [nz][2 ny][2 nx]
    CUtensorMap conv_map;   // tensor map of the array k_conv transforms in place (W1 in 2-D, W2 in 3-D)
    float *abl[3] = {nullptr, nullptr, nullptr};
    double *norms = nullptr, *history = nullptr;
    int hist_cap = 0;
    unsigned int *maxbits = nullptr;
    Ctl *h_ctl = nullptr;        // pinned, 4 slots
    double *h_hist = nullptr;    // pinned staging
    cudaEvent_t ev[2] = {nullptr, nullptr}, ev_t0 = nullptr, ev_t1 = nullptr;
    size_t dev_bytes = 0;
    int graph_batch = 16;
    int scheme = TBS_SCHEME_BORN;
    int boundary = TBS_BOUNDARY_PAD;
    int crit_row = -1;
    long long launches = 0;
    double loop_ms = 0;
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
    if (e == cudaSuccess) p->dev_bytes += count * sizeof(T);
    return e;
}

bool pow2(int v) { return v > 0 && (v & (v - 1)) == 0; }
inline unsigned nblk(long long n, int b) { return (unsigned)((n + b - 1) / b); }

void fill_row_args(tbs_plan *pl, Freq &f, RowArgs &a, const float2 *src, float src_scale, int do_fwd) {
    a.W = pl->W1;
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
    a.norms = pl->norms;
    a.history = pl->history;
    a.ctl = f.ctl;
    a.lut = Luts{pl->lutA[0], pl->lutB[0], pl->lutC[0], pl->lutAB[0]};
}

// Column / plane passes of one term (K2 in 2-D; y-forward, z-conv, y-inverse in 3-D).
cudaError_t launch_mid_passes(tbs_plan *pl, Freq &f, cudaStream_t st, int which = -1) {
    const int nx = pl->n[0], ny = pl->n[1], nz = pl->n[2];
    const long long mx = 2LL * nx, my = 2LL * ny;
    ColArgs a;
    memset(&a, 0, sizeof a);
    a.ctl = f.ctl;
    a.inv_e = (float)(1.0 / pl->damping);
    a.kabs = f.kabs;
    a.masked = pl->boundary == TBS_BOUNDARY_PERIODIC;
    a.inner_len = (int)mx;
    cudaError_t e = cudaSuccess;
    if (pl->ndim == 2) {
        a.in = pl->W1; a.out = pl->W1;
        a.lut = Luts{pl->lutA[1], pl->lutB[1], pl->lutC[1], pl->lutAB[1]};
        a.in_line_stride = a.out_line_stride = mx;
        a.p2_line = (const float2 *)f.p2[1]; a.p2_inner = f.p2[0]; a.p2_outer = nullptr;
        if (which < 0 || which == 0) e = launch_conv(ny, a, &pl->conv_map, 1, st);
        return e;
    }
    // y forward: W1[z][y][kx] -> W2[z][ky][kx]
    if (which < 0 || which == 0) {
        a.in = pl->W1; a.out = pl->W2;
        a.lut = Luts{pl->lutA[1], pl->lutB[1], pl->lutC[1], pl->lutAB[1]};
        a.in_line_stride = mx; a.out_line_stride = mx;
        a.in_outer_stride = (long long)ny * mx; a.out_outer_stride = my * mx;
        e = launch_col<MODE_FWD>(ny, a, nz, st);
        if (e != cudaSuccess) return e;
    }
    // z convolution, in place on W2; lines (ky, kx), outer = ky
    if (which < 0 || which == 1) {
        a.in = pl->W2; a.out = pl->W2;
        a.lut = Luts{pl->lutA[2], pl->lutB[2], pl->lutC[2], pl->lutAB[2]};
        a.in_line_stride = a.out_line_stride = my * mx;
        a.in_outer_stride = a.out_outer_stride = mx;
        a.p2_line = (const float2 *)f.p2[2]; a.p2_inner = f.p2[0]; a.p2_outer = f.p2[1];
        e = launch_conv(nz, a, &pl->conv_map, (int)my, st);
        if (e != cudaSuccess) return e;
    }
    // y inverse: W2[z][ky][kx] -> W1[z][y][kx]
    if (which < 0 || which == 2) {
        a.in = pl->W2; a.out = pl->W1;
        a.lut = Luts{pl->lutA[1], pl->lutB[1], pl->lutC[1], pl->lutAB[1]};
        a.in_line_stride = mx; a.out_line_stride = mx;
        a.in_outer_stride = my * mx; a.out_outer_stride = (long long)ny * mx;
        a.p2_line = nullptr; a.p2_inner = nullptr; a.p2_outer = nullptr;
        e = launch_col<MODE_INV>(ny, a, nz, st);
    }
    return e;
}

int mid_launches(const tbs_plan *pl) { return pl->ndim == 2 ? 1 : 3; }

cudaError_t launch_term(tbs_plan *pl, Freq &f, cudaStream_t st, int do_fwd = 1) {
    cudaError_t e = launch_mid_passes(pl, f, st);
    if (e != cudaSuccess) return e;
    RowArgs r;
    fill_row_args(pl, f, r, nullptr, 0.f, do_fwd);
    return launch_row<false>(pl->n[0], r, st);
}

// Green's-spectrum axis tables of one frequency, in the order each kernel reads them (setup_kernels.cuh).
void fill_axis_tables(tbs_plan *pl, Freq &f) {
    for (int a = 0; a < pl->ndim; ++a) {
        int r1, r2, rl;
        radices_of(pl->n[a], r1, r2, rl);
        k_axis_table<<<nblk(2 * pl->n[a], 256), 256>>>(f.p2[a], pl->n[a], r1, r2, rl, pl->dx, f.k0,
                                                        a == 0 || a == pl->ndim - 1,
                                                        a == pl->ndim - 1 ? 1.0 / pl->damping : 1.0,
                                                        pl->boundary == TBS_BOUNDARY_PERIODIC);
    }
}

cudaError_t set_kernel_attrs(tbs_plan *pl) {
    ColArgs ca; memset(&ca, 0, sizeof ca);
    RowArgs ra; memset(&ra, 0, sizeof ra);
    cudaError_t e;
    if ((e = launch_row<true>(pl->n[0], ra, 0, true)) != cudaSuccess) return e;
    if ((e = launch_row<false>(pl->n[0], ra, 0, true)) != cudaSuccess) return e;
    if (pl->ndim == 2) return launch_conv(pl->n[1], ca, nullptr, 1, 0, true);
    if ((e = launch_col<MODE_FWD>(pl->n[1], ca, 1, 0, true)) != cudaSuccess) return e;
    if ((e = launch_col<MODE_INV>(pl->n[1], ca, 1, 0, true)) != cudaSuccess) return e;
    return launch_conv(pl->n[2], ca, nullptr, 1, 0, true);
}

tbs_status ensure_history(tbs_plan *pl, int max_terms) {
    if (max_terms + 1 <= pl->hist_cap) return TBS_OK;
    if (pl->norms) { cudaFree(pl->norms); cudaFree(pl->history); cudaFreeHost(pl->h_hist); }
    pl->norms = nullptr; pl->history = nullptr; pl->h_hist = nullptr;
    const int cap = max_terms + 1;
    CU(pl, cudaMalloc((void **)&pl->norms, sizeof(double) * 2 * cap));
    CU(pl, cudaMalloc((void **)&pl->history, sizeof(double) * cap));
    CU(pl, cudaMallocHost((void **)&pl->h_hist, sizeof(double) * cap));
    pl->hist_cap = cap;
    return TBS_OK;
}

void destroy_graphs(tbs_plan *pl) {
    for (auto &f : pl->fr) {
        if (f.graph) cudaGraphExecDestroy(f.graph);
        f.graph = nullptr;
        f.graph_batch = 0;
    }
}

}  // namespace

extern "C" {

const char *tbs_version(void) { return "tbs-b200 0.1 (sm_100a)"; }

const char *tbs_last_error(const tbs_plan *plan) { return plan ? plan->err.c_str() : "null plan"; }

size_t tbs_plan_workspace_bytes(const tbs_plan *plan) { return plan ? plan->dev_bytes : 0; }

int64_t tbs_last_launch_count(const tbs_plan *plan) { return plan ? plan->launches : 0; }
double tbs_last_loop_ms(const tbs_plan *plan) { return plan ? plan->loop_ms : 0.0; }

tbs_status tbs_set_graph_batch(tbs_plan *plan, int terms_per_graph) {
    if (!plan || terms_per_graph < 0 || terms_per_graph > 1024) return TBS_ERR_INVALID_ARG;
    plan->graph_batch = terms_per_graph;
    destroy_graphs(plan);
    return TBS_OK;
}

void tbs_plan_destroy(tbs_plan *pl) {
    if (!pl) return;
    destroy_graphs(pl);
    for (auto &f : pl->fr) {
        cudaFree(f.V); cudaFree(f.S); cudaFree(f.p); cudaFree(f.ctl); cudaFree(f.ucbs);
        for (int a = 0; a < 3; ++a) cudaFree(f.p2[a]);
    }
    for (int a = 0; a < 3; ++a) { cudaFree(pl->lutA[a]); cudaFree(pl->lutB[a]); cudaFree(pl->lutC[a]); cudaFree(pl->lutAB[a]); }
    cudaFree(pl->W1); cudaFree(pl->W2);
    for (int a = 0; a < 3; ++a) cudaFree(pl->abl[a]);
    cudaFree(pl->norms); cudaFree(pl->history); cudaFree(pl->maxbits);
    if (pl->h_ctl) cudaFreeHost(pl->h_ctl);
    if (pl->h_hist) cudaFreeHost(pl->h_hist);
    for (int i = 0; i < 2; ++i) if (pl->ev[i]) cudaEventDestroy(pl->ev[i]);
    if (pl->ev_t0) cudaEventDestroy(pl->ev_t0);
    if (pl->ev_t1) cudaEventDestroy(pl->ev_t1);
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
    tbs_status st = TBS_OK;
    auto build = [&]() -> tbs_status {
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
            k_stage_lut_ab<<<nblk(N, 256), 256>>>(pl->lutAB[a], N, r1);
            if (r2 > 0) {
                CU(pl, dmalloc(pl, &pl->lutC[a], N / r1));
                k_stage_lut<<<nblk(N / r1, 256), 256>>>(pl->lutC[a], N / r1, r2, 0);
            }
        }
        const long long rows = (long long)pl->n[1] * pl->n[2];
        CU(pl, dmalloc(pl, &pl->W1, (size_t)(rows * 2 * pl->n[0])));
        if (ndim == 3) CU(pl, dmalloc(pl, &pl->W2, (size_t)((long long)pl->n[2] * 2 * pl->n[1] * 2 * pl->n[0])));
        {
            const long long mx = 2LL * pl->n[0], my = 2LL * pl->n[1];
            if (ndim == 2) CU(pl, make_conv_tensor_map(&pl->conv_map, pl->W1, mx, pl->n[1], mx, conv_tile_width(pl->n[1])));
            else CU(pl, make_conv_tensor_map(&pl->conv_map, pl->W2, my * mx, pl->n[2], my * mx, conv_tile_width(pl->n[2])));
        }
        for (int a = 0; a < ndim; ++a) {
            CU(pl, dmalloc(pl, &pl->abl[a], pl->n[a]));
            k_abl_window<<<nblk(pl->n[a], 256), 256>>>(pl->abl[a], pl->n[a], 0, 0.0);
        }
        CU(pl, dmalloc(pl, &pl->maxbits, 1));
        CU(pl, cudaMallocHost((void **)&pl->h_ctl, sizeof(Ctl) * 4));
        for (int i = 0; i < 2; ++i) CU(pl, cudaEventCreateWithFlags(&pl->ev[i], cudaEventDisableTiming));
        CU(pl, cudaEventCreate(&pl->ev_t0));
        CU(pl, cudaEventCreate(&pl->ev_t1));
        for (int i = 0; i < nfreq; ++i) {
            Freq &f = pl->fr[i];
            f.f = f_hz[i];
            f.omega = 2.0 * kPi * f.f;
            f.k0 = f.omega / c0;
            CU(pl, dmalloc(pl, &f.V, (size_t)pl->npts));
            CU(pl, dmalloc(pl, &f.S, (size_t)pl->npts));
            CU(pl, dmalloc(pl, &f.p, (size_t)pl->npts));
            CU(pl, dmalloc(pl, &f.ctl, 1));
            for (int a = 0; a < ndim; ++a) CU(pl, dmalloc(pl, &f.p2[a], 2 * pl->n[a]));
            fill_axis_tables(pl, f);
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
    if (!pl || !(alpha0_si >= 0.0)) return TBS_ERR_INVALID_ARG;
    if (alpha0_si > 0.0 && (!(nu > 0.0) || nu > 2.0 || fabs(nu - 1.0) < 1e-9))
        return fail(pl, TBS_ERR_INVALID_ARG, "power-law exponent must lie in (0, 2] and differ from 1 (PAPER.md:53)");
    for (auto &f : pl->fr) {
        if (alpha0_si == 0.0) {
            f.kabs = KAbs{0.f, 0.f, 0.f, 0.f};
            f.have_V = false;  // the spatial potential has to be set again
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
    CU(pl, cudaDeviceSynchronize());
    return TBS_OK;
}

tbs_status tbs_set_boundary(tbs_plan *pl, int boundary) {
    if (!pl || (boundary != TBS_BOUNDARY_PAD && boundary != TBS_BOUNDARY_PERIODIC)) return TBS_ERR_INVALID_ARG;
    pl->boundary = boundary;
    for (auto &f : pl->fr) fill_axis_tables(pl, f);
    destroy_graphs(pl);  // the captured launches carry the normalisation
    CU(pl, cudaDeviceSynchronize());
    return TBS_OK;
}

tbs_status tbs_set_criterion(tbs_plan *pl, int criterion, int row) {
    if (!pl || (criterion != TBS_CRIT_L2_GRID && criterion != TBS_CRIT_L1_ROW)) return TBS_ERR_INVALID_ARG;
    const int rows = pl->n[1] * (pl->ndim == 3 ? pl->n[2] : 1);
    if (criterion == TBS_CRIT_L1_ROW && (row < 0 || row >= rows)) return fail(pl, TBS_ERR_INVALID_ARG, "row outside the grid");
    pl->crit_row = criterion == TBS_CRIT_L1_ROW ? row : -1;
    destroy_graphs(pl);
    return TBS_OK;
}

tbs_status tbs_set_scheme(tbs_plan *pl, int scheme) {
    if (!pl || (scheme != TBS_SCHEME_BORN && scheme != TBS_SCHEME_CBS)) return TBS_ERR_INVALID_ARG;
    if (scheme == TBS_SCHEME_CBS)
        for (auto &f : pl->fr)
            if (!f.ucbs) CU(pl, dmalloc(pl, &f.ucbs, (size_t)pl->npts));
    if (scheme != pl->scheme) destroy_graphs(pl);  // the captured launches carry the scheme
    pl->scheme = scheme;
    return TBS_OK;
}

tbs_status tbs_set_abl(tbs_plan *pl, int cells, double zeta_half_mu) {
    if (!pl || cells < 0) return TBS_ERR_INVALID_ARG;
    for (int a = 0; a < pl->ndim; ++a)
        if (2 * cells > pl->n[a]) return fail(pl, TBS_ERR_INVALID_ARG, "ABL wider than half the grid");
    for (int a = 0; a < pl->ndim; ++a)
        k_abl_window<<<nblk(pl->n[a], 256), 256>>>(pl->abl[a], pl->n[a], cells, zeta_half_mu);
    CU(pl, cudaDeviceSynchronize());
    return TBS_OK;
}

tbs_status tbs_set_medium(tbs_plan *pl, const float *c, const float *rho, const float *alpha0_map,
                          double alpha0_db, double y, double beta, double rho0, void *stream) {
    if (!pl || !c) return TBS_ERR_INVALID_ARG;
    const bool absorbing = alpha0_map != nullptr || alpha0_db != 0.0;
    if (absorbing && fabs(y - 1.0) < 1e-9) return fail(pl, TBS_ERR_INVALID_ARG, "y = 1 is excluded (PAPER.md:53)");
    if (!(rho0 > 0) && !rho) return fail(pl, TBS_ERR_INVALID_ARG, "rho0 must be positive");
    (void)rho;  // density does not enter V; rho0 feeds xi of the harmonic source
    cudaStream_t st = (cudaStream_t)stream;
    pl->beta = beta;
    pl->rho0 = rho0;
    for (auto &f : pl->fr) {
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
    cudaStream_t st = (cudaStream_t)stream;
    // stage through W1 (>= 2 n complex = 4 n floats): c at [0, n), alpha0 map at [n, 2n)
    float *dc = (float *)pl->W1;
    float *da = alpha0_map ? dc + pl->npts : nullptr;
    CU(pl, cudaMemcpyAsync(dc, c, sizeof(float) * pl->npts, cudaMemcpyHostToDevice, st));
    if (alpha0_map) CU(pl, cudaMemcpyAsync(da, alpha0_map, sizeof(float) * pl->npts, cudaMemcpyHostToDevice, st));
    return tbs_set_medium(pl, dc, rho ? dc : nullptr, da, alpha0_db, y, beta, rho0, stream);
}

tbs_status tbs_set_potential(tbs_plan *pl, int ifreq, const float *V, void *stream) {
    if (!pl || !V || ifreq < 0 || ifreq >= (int)pl->fr.size()) return TBS_ERR_INVALID_ARG;
    cudaStream_t st = (cudaStream_t)stream;
    Freq &f = pl->fr[ifreq];
    k_scale_complex<<<nblk(pl->npts, 256), 256, 0, st>>>(f.V, (const float2 *)V, 1.0 / (f.k0 * f.k0), pl->npts);
    CU(pl, cudaGetLastError());
    CU(pl, cudaStreamSynchronize(st));
    f.have_V = true;
    return TBS_OK;
}

tbs_status tbs_set_source(tbs_plan *pl, int n_src, const double *pos_m, const float *amp, void *stream) {
    if (!pl || n_src < 1 || !pos_m || !amp) return TBS_ERR_INVALID_ARG;
    for (int j = 0; j < n_src; ++j)
        for (int a = 0; a < pl->ndim; ++a) {
            const double g = pos_m[(size_t)j * pl->ndim + a] / pl->dx;
            if (!(g >= 0.0) || g > (double)(pl->n[a] - 1))
                return fail(pl, TBS_ERR_INVALID_ARG, "source %d lies outside the grid", j);
        }
    cudaStream_t st = (cudaStream_t)stream;
    double *dpos = nullptr;
    float2 *damp = nullptr;
    const size_t nf = pl->fr.size();
    CU(pl, cudaMalloc((void **)&dpos, sizeof(double) * n_src * pl->ndim));
    cudaError_t e = cudaMalloc((void **)&damp, sizeof(float2) * n_src * nf);
    if (e != cudaSuccess) { cudaFree(dpos); return fail(pl, TBS_ERR_ALLOC, "cudaMalloc(amp)"); }
    cudaMemcpyAsync(dpos, pos_m, sizeof(double) * n_src * pl->ndim, cudaMemcpyHostToDevice, st);
    cudaMemcpyAsync(damp, amp, sizeof(float2) * n_src * nf, cudaMemcpyHostToDevice, st);
    for (size_t i = 0; i < nf; ++i) {
        Freq &f = pl->fr[i];
        cudaMemsetAsync(f.S, 0, sizeof(float2) * pl->npts, st);
        k_deposit<<<nblk((long long)n_src << pl->ndim, 128), 128, 0, st>>>(f.S, dpos, damp + i * n_src, n_src,
                                                                            pl->ndim, pl->n[0], pl->n[1], pl->n[2], pl->dx);
        f.have_S = true;
    }
    e = cudaStreamSynchronize(st);
    cudaFree(dpos);
    cudaFree(damp);
    CU(pl, e);
    CU(pl, cudaGetLastError());
    return TBS_OK;
}

tbs_status tbs_set_source_field(tbs_plan *pl, int ifreq, const float *S, void *stream) {
    if (!pl || !S || ifreq < 0 || ifreq >= (int)pl->fr.size()) return TBS_ERR_INVALID_ARG;
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
