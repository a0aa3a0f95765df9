/*
 * oracle/tbs_ref.c -- TEST INFRASTRUCTURE, NOT THE PRODUCT.
 *
 * Plain, slow, obviously-correct CPU complex128 implementation of the traditional Born
 * series (TBS) solve of the inhomogeneous Helmholtz equation, written from the paper
 * (arxiv 2507.13754, /root/reference/PAPER.md; citations below are PAPER.md line numbers).
 * Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs
 * may load this library.  It shares no source, header, table or constant generator with
 * the CUDA library under paper_2507_13754_b200/csrc/.
 *
 * What it computes (the readings are listed in DESIGN.md):
 *   k0 = 2 pi f / c0,  eps = damping * k0^2
 *   ghat(p) = 1 / (|p|^2 - k0^2 - i eps)  on the padded M^d grid
 *   G x  = crop( IDFT_M( ghat . DFT_M( zero-pad(x) ) ) )
 *   u_0 = A.(G S),  u_{n+1} = A.G(V.u_n),  p = sum_n u_n                  (Eq.18,
 *                                                                          160 Eq.19, 164 Eq.20)
 *   r_n = ||u_n||_2 / ||p_n||_2, stop at the first n>=1 with r_n < tol
 *
 * The FFT is a hand-written iterative radix-2 transform (naive O(n^2) DFT for lengths that
 * are not a power of two); no blocking, pruning or fusion: the padded array is materialised
 * and every line of it is transformed.  OpenMP is used only over independent 1-D lines.
 *
 * Parity pins (tests/test_oracle_*.py, -m "not gpu"): printed constants (P1), damped
 * Hankel / spherical closed forms (P2), lossless line-source Hankel sum with ABL (P3),
 * exact diagonal special case (P4), brute-force first term (P5), dense Lippmann-Schwinger
 * solve (P6), invariants (P7), FFT vs naive DFT (P8).
 * The Python side (tbs_ref.py) adds, on top of apply_G: the harmonic sources of Eqs. 28b-28e (pinned by
 * a Westervelt sum-frequency projection), the convergent Born series, Algorithm 1 as printed (periodic
 * grid, Eq. 30) and the k-space multiplier potential of Eq. 24 (tests/test_oracle_pins_d.py).
 * parity unpinned: the paper's k-Wave agreement figures (they need k-Wave).  The iteration
 * counts of Table 3 are checked on the GPU path, whole table within 7 %
 * (tests/test_gpu_paper_mode.py); the oracle itself is not run at 4096^2.
 */
#include <complex.h>
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

typedef double complex cplx;

#define TBS_REF_OK 0
#define TBS_REF_NOT_CONVERGED 1
#define TBS_REF_ERR_INVALID_ARG (-1)
#define TBS_REF_ERR_DIVERGED (-5)
#define TBS_REF_ERR_ALLOC (-6)

static const double PI = 3.14159265358979323846264338327950288;

int tbs_ref_num_threads(void) {
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}

/* ---- 1-D DFT ------------------------------------------------------------------------
 * X[k] = sum_j x[j] exp(sign * 2 pi i j k / n), unnormalised, sign = -1 forward, +1 inverse. */
static void dft_naive(cplx *x, int n, int sign) {
    cplx *t = (cplx *)malloc(sizeof(cplx) * (size_t)n);
    for (int k = 0; k < n; ++k) {
        cplx acc = 0.0;
        for (int j = 0; j < n; ++j) {
            long jk = ((long)j * (long)k) % n;
            double ang = sign * 2.0 * PI * (double)jk / (double)n;
            acc += x[j] * (cos(ang) + I * sin(ang));
        }
        t[k] = acc;
    }
    memcpy(x, t, sizeof(cplx) * (size_t)n);
    free(t);
}

static void fft_radix2(cplx *x, int n, int sign) {
    /* bit-reversal permutation */
    for (int i = 1, j = 0; i < n; ++i) {
        int bit = n >> 1;
        for (; j & bit; bit >>= 1) j ^= bit;
        j ^= bit;
        if (i < j) { cplx t = x[i]; x[i] = x[j]; x[j] = t; }
    }
    /* decimation-in-time butterflies; each twiddle is evaluated directly (no recurrence) */
    for (int len = 2; len <= n; len <<= 1) {
        int half = len >> 1;
        for (int j = 0; j < half; ++j) {
            double ang = sign * 2.0 * PI * (double)j / (double)len;
            cplx w = cos(ang) + I * sin(ang);
            for (int i = j; i < n; i += len) {
                cplx a = x[i], b = x[i + half] * w;
                x[i] = a + b;
                x[i + half] = a - b;
            }
        }
    }
}

void tbs_ref_fft1d(double *x_reim, int n, int sign) {
    cplx *x = (cplx *)x_reim;
    if (n <= 1) return;
    if ((n & (n - 1)) == 0) fft_radix2(x, n, sign);
    else dft_naive(x, n, sign);
}

/* Transform every line along `axis` (0 = x fastest, 1 = y, 2 = z) of a row-major array
 * with dims d[0]=nx, d[1]=ny, d[2]=nz. */
static void fft_axis(cplx *a, const int64_t d[3], int axis, int sign) {
    int64_t len = d[axis];
    int64_t stride = 1;
    for (int i = 0; i < axis; ++i) stride *= d[i];
    int64_t total = d[0] * d[1] * d[2];
    int64_t nlines = total / len;
#pragma omp parallel
    {
        cplx *buf = (cplx *)malloc(sizeof(cplx) * (size_t)len);
#pragma omp for schedule(static)
        for (int64_t l = 0; l < nlines; ++l) {
            /* line l: inner index (below the axis) and outer index (above it) */
            int64_t inner = l % stride, outer = l / stride;
            cplx *base = a + outer * stride * len + inner;
            for (int64_t j = 0; j < len; ++j) buf[j] = base[j * stride];
            tbs_ref_fft1d((double *)buf, (int)len, sign);
            for (int64_t j = 0; j < len; ++j) base[j * stride] = buf[j];
        }
        free(buf);
    }
}

/* ---- Green's spectrum; Alg. 1 l.9-12 ----------------
 * ghat[m] = 1/(|p_m|^2 - k0^2 - i eps); p component i = 2 pi mt/(M dx), mt = m for m < M/2,
 * m - M otherwise (the paper builds the same thing on a centred grid and fftShifts it,
 * PAPER.md:346).  Written as ((p2-k0^2) + i eps)/((p2-k0^2)^2 + eps^2) exactly as Alg. 1. */
int tbs_ref_green_spectrum(int ndim, const int32_t M[3], double dx, double k0, double eps,
                           double *ghat_reim) {
    if (ndim < 1 || ndim > 3 || dx <= 0) return TBS_REF_ERR_INVALID_ARG;
    int64_t mx = M[0], my = ndim > 1 ? M[1] : 1, mz = ndim > 2 ? M[2] : 1;
    cplx *g = (cplx *)ghat_reim;
    for (int64_t iz = 0; iz < mz; ++iz)
        for (int64_t iy = 0; iy < my; ++iy)
            for (int64_t ix = 0; ix < mx; ++ix) {
                double fx = (double)(ix < (mx + 1) / 2 ? ix : ix - mx);
                double fy = (double)(iy < (my + 1) / 2 ? iy : iy - my);
                double fz = (double)(iz < (mz + 1) / 2 ? iz : iz - mz);
                double px = 2.0 * PI * fx / ((double)mx * dx);
                double py = ndim > 1 ? 2.0 * PI * fy / ((double)my * dx) : 0.0;
                double pz = ndim > 2 ? 2.0 * PI * fz / ((double)mz * dx) : 0.0;
                double a = px * px + py * py + pz * pz - k0 * k0;
                double D = a * a + eps * eps;
                g[(iz * my + iy) * mx + ix] = a / D + I * (eps / D);
            }
    return TBS_REF_OK;
}

/* ---- Potential from the medium maps (reading A6 of SURVEY.md 8(c)) -------------------
 * alpha = alpha0_SI * omega^y (Eq.3), alpha0_SI [Np (rad/s)^-y m^-1] =
 * alpha0_dB * 100 / 8.685889638 / (2 pi 1e6)^y;
 * ktilde = omega/c + alpha*tan(pi y/2) + i*alpha  (plane-wave dispersion relation of Eq. 7,
 * PAPER.md:72, with tau, eta of PAPER.md:58, to first order in alpha/k);
 * V = ktilde^2 - k0^2 - i eps.  alpha0_map may be NULL (scalar used). */
int tbs_ref_potential(int64_t n, const double *c, const double *alpha0_db_map,
                      double alpha0_db, double y, double f_hz, double c0, double damping,
                      double *V_reim) {
    if (n <= 0 || !c || !V_reim || f_hz <= 0 || c0 <= 0) return TBS_REF_ERR_INVALID_ARG;
    double omega = 2.0 * PI * f_hz;
    double k0 = omega / c0;
    double eps = damping * k0 * k0;
    cplx *V = (cplx *)V_reim;
    for (int64_t i = 0; i < n; ++i) {
        double a0 = alpha0_db_map ? alpha0_db_map[i] : alpha0_db;
        cplx kt = omega / c[i];
        if (a0 != 0.0) {
            double a0_si = a0 * 100.0 / 8.685889638 / pow(2.0 * PI * 1.0e6, y);
            double alpha = a0_si * pow(omega, y);
            kt += alpha * tan(PI * y / 2.0) + I * alpha;
        }
        V[i] = kt * kt - k0 * k0 - I * eps;
    }
    return TBS_REF_OK;
}

/* ---- Source deposition (reading A9) --------------------------------------------------
 * S(r) = sum_j a_j w_j(r), multilinear (cloud-in-cell) weights that sum to 1; a point on a
 * node gives the paper's single-pixel source.  pos in metres, the centre
 * of cell (0,0,0) is r = 0.  Points outside [0, N-1] cells are an error. */
int tbs_ref_deposit(int ndim, const int32_t N[3], double dx, int n_src, const double *pos,
                    const double *amp_reim, double *S_reim) {
    if (ndim < 1 || ndim > 3) return TBS_REF_ERR_INVALID_ARG;
    int64_t nx = N[0], ny = ndim > 1 ? N[1] : 1, nz = ndim > 2 ? N[2] : 1;
    int64_t dims[3] = {nx, ny, nz};
    cplx *S = (cplx *)S_reim;
    const cplx *amp = (const cplx *)amp_reim;
    memset(S, 0, sizeof(cplx) * (size_t)(nx * ny * nz));
    for (int j = 0; j < n_src; ++j) {
        int64_t i0[3] = {0, 0, 0};
        double fr[3] = {0, 0, 0};
        for (int a = 0; a < ndim; ++a) {
            double g = pos[(int64_t)j * ndim + a] / dx;
            if (g < 0.0 || g > (double)(dims[a] - 1)) return TBS_REF_ERR_INVALID_ARG;
            double fl = floor(g);
            if (fl > (double)(dims[a] - 2) && dims[a] > 1) fl = (double)(dims[a] - 2);
            i0[a] = (int64_t)fl;
            fr[a] = g - fl;
        }
        for (int cz = 0; cz < (ndim > 2 ? 2 : 1); ++cz)
            for (int cy = 0; cy < (ndim > 1 ? 2 : 1); ++cy)
                for (int cx = 0; cx < 2; ++cx) {
                    double w = (cx ? fr[0] : 1.0 - fr[0]);
                    if (ndim > 1) w *= (cy ? fr[1] : 1.0 - fr[1]);
                    if (ndim > 2) w *= (cz ? fr[2] : 1.0 - fr[2]);
                    if (w == 0.0) continue;
                    int64_t ix = i0[0] + cx, iy = i0[1] + cy, iz = i0[2] + cz;
                    if (ix >= nx || iy >= ny || iz >= nz) continue;
                    S[(iz * ny + iy) * nx + ix] += amp[j] * w;
                }
    }
    return TBS_REF_OK;
}

/* ---- Absorbing-layer window, Eq.29 (reading A4) ----------------------
 * One axis: a[i] = 1/(1+exp(-zeta*(x - mu/2))) for x = distance from the nearer outer edge
 * (in cells, cell i has x = i) while x < cells, 1 elsewhere; zeta*mu/2 = zeta_half_mu
 * (paper: 21.48 Np/cm * 0.45 cm / 2 = 9.666). */
int tbs_ref_abl_window(int n, int cells, double zeta_half_mu, double *a) {
    if (n <= 0 || cells < 0 || 2 * cells > n) return TBS_REF_ERR_INVALID_ARG;
    for (int i = 0; i < n; ++i) {
        int x = i < n - 1 - i ? i : n - 1 - i;
        if (cells > 0 && x < cells) {
            double zeta = 2.0 * zeta_half_mu / (double)cells; /* per cell */
            a[i] = 1.0 / (1.0 + exp(-zeta * ((double)x - 0.5 * (double)cells)));
        } else {
            a[i] = 1.0;
        }
    }
    return TBS_REF_OK;
}

/* ---- G x, PAPER.md:154 and 352 ("ifft(G x fft(S))") -----------------------------------
 * pad = 2: zero-pad N -> M = 2N per axis (linear convolution, BASELINE.json north_star);
 * pad = 1: periodic (the paper's own variant; used by pin P4 only).
 * ghat has pad*N points per axis. */
int tbs_ref_apply_G(int ndim, const int32_t N[3], int pad, const double *ghat_reim,
                    const double *x_reim, double *out_reim) {
    if (ndim < 1 || ndim > 3 || (pad != 1 && pad != 2)) return TBS_REF_ERR_INVALID_ARG;
    int64_t n[3] = {N[0], ndim > 1 ? N[1] : 1, ndim > 2 ? N[2] : 1};
    int64_t m[3] = {n[0] * pad, ndim > 1 ? n[1] * pad : 1, ndim > 2 ? n[2] * pad : 1};
    int64_t mt = m[0] * m[1] * m[2];
    const cplx *x = (const cplx *)x_reim, *g = (const cplx *)ghat_reim;
    cplx *out = (cplx *)out_reim;
    cplx *w = (cplx *)calloc((size_t)mt, sizeof(cplx));
    if (!w) return TBS_REF_ERR_ALLOC;
    /* Z: place the array at indices 0..N-1 of a zero M^d array */
    for (int64_t iz = 0; iz < n[2]; ++iz)
        for (int64_t iy = 0; iy < n[1]; ++iy)
            for (int64_t ix = 0; ix < n[0]; ++ix)
                w[(iz * m[1] + iy) * m[0] + ix] = x[(iz * n[1] + iy) * n[0] + ix];
    for (int a = 0; a < ndim; ++a) fft_axis(w, m, a, -1);
#pragma omp parallel for schedule(static)
    for (int64_t i = 0; i < mt; ++i) w[i] *= g[i];
    for (int a = 0; a < ndim; ++a) fft_axis(w, m, a, +1);
    double inv = 1.0 / (double)mt;
    /* C: keep indices 0..N-1; the IDFT carries 1/M^d */
    for (int64_t iz = 0; iz < n[2]; ++iz)
        for (int64_t iy = 0; iy < n[1]; ++iy)
            for (int64_t ix = 0; ix < n[0]; ++ix)
                out[(iz * n[1] + iy) * n[0] + ix] = w[(iz * m[1] + iy) * m[0] + ix] * inv;
    free(w);
    return TBS_REF_OK;
}

static void apply_window(int ndim, const int64_t n[3], const double *ax, const double *ay,
                         const double *az, cplx *u) {
    if (!ax && !ay && !az) return;
    for (int64_t iz = 0; iz < n[2]; ++iz)
        for (int64_t iy = 0; iy < n[1]; ++iy)
            for (int64_t ix = 0; ix < n[0]; ++ix) {
                double a = (ax ? ax[ix] : 1.0);
                if (ndim > 1 && ay) a *= ay[iy];
                if (ndim > 2 && az) a *= az[iz];
                u[(iz * n[1] + iy) * n[0] + ix] *= a;
            }
}

/* ---- The series, Eq.18 in term form ---------------------------------------
 * u_0 = A.(G S); p_0 = u_0; u_{n+1} = A.G(V.u_n); p_{n+1} = p_n + u_{n+1};
 * history[n] = ||u_n||_2/||p_n||_2 (history[0] = 1).  Stops at the first n >= 1 with
 * history[n] < tol (TBS_REF_OK) or at n = max_terms (TBS_REF_NOT_CONVERGED); a non-finite
 * norm returns TBS_REF_ERR_DIVERGED.  ax/ay/az: per-axis ABL windows or NULL (A == 1).
 * u_last (optional) receives the last term added. */
int tbs_ref_solve(int ndim, const int32_t N[3], int pad, const double *ghat_reim,
                  const double *V_reim, const double *S_reim, const double *ax,
                  const double *ay, const double *az, int max_terms, double tol,
                  double *p_reim, double *history, int32_t *n_terms, double *u_last_reim) {
    if (ndim < 1 || ndim > 3 || max_terms < 0) return TBS_REF_ERR_INVALID_ARG;
    int64_t n[3] = {N[0], ndim > 1 ? N[1] : 1, ndim > 2 ? N[2] : 1};
    int64_t nt = n[0] * n[1] * n[2];
    const cplx *V = (const cplx *)V_reim;
    cplx *p = (cplx *)p_reim;
    cplx *u = (cplx *)malloc(sizeof(cplx) * (size_t)nt);
    cplx *w = (cplx *)malloc(sizeof(cplx) * (size_t)nt);
    if (!u || !w) { free(u); free(w); return TBS_REF_ERR_ALLOC; }
    int rc = tbs_ref_apply_G(ndim, N, pad, ghat_reim, S_reim, (double *)u);
    if (rc != TBS_REF_OK) { free(u); free(w); return rc; }
    apply_window(ndim, n, ax, ay, az, u);
    memcpy(p, u, sizeof(cplx) * (size_t)nt);
    history[0] = 1.0;
    int term = 0;
    int status = (max_terms == 0) ? TBS_REF_NOT_CONVERGED : TBS_REF_OK;
    while (term < max_terms) {
        for (int64_t i = 0; i < nt; ++i) w[i] = V[i] * u[i];
        rc = tbs_ref_apply_G(ndim, N, pad, ghat_reim, (double *)w, (double *)u);
        if (rc != TBS_REF_OK) { status = rc; break; }
        apply_window(ndim, n, ax, ay, az, u);
        double uu = 0.0, pp = 0.0;
        for (int64_t i = 0; i < nt; ++i) {
            p[i] += u[i];
            uu += creal(u[i]) * creal(u[i]) + cimag(u[i]) * cimag(u[i]);
            pp += creal(p[i]) * creal(p[i]) + cimag(p[i]) * cimag(p[i]);
        }
        ++term;
        double r = sqrt(uu) / sqrt(pp);
        history[term] = r;
        if (!isfinite(r)) { status = TBS_REF_ERR_DIVERGED; break; }
        if (r < tol) { status = TBS_REF_OK; break; }
        status = TBS_REF_NOT_CONVERGED;
    }
    *n_terms = term;
    if (u_last_reim) memcpy(u_last_reim, u, sizeof(cplx) * (size_t)nt);
    free(u);
    free(w);
    return status;
}

/* ---- Second-harmonic source, Eq.28b with xi of PAPER.md:117 ----------------
 * S2(r) = -xi (2 omega1)^2 (1/2) p1(r)^2,  xi = beta/(rho0 c0^4), beta = 1 + B/2A. */
int tbs_ref_second_harmonic_source(int64_t n, const double *p1_reim, double beta, double rho0,
                                   double c0, double f1_hz, double *S2_reim) {
    if (n <= 0 || rho0 <= 0 || c0 <= 0) return TBS_REF_ERR_INVALID_ARG;
    const cplx *p1 = (const cplx *)p1_reim;
    cplx *S2 = (cplx *)S2_reim;
    double xi = beta / (rho0 * c0 * c0 * c0 * c0);
    double w2 = 2.0 * (2.0 * PI * f1_hz);
    for (int64_t i = 0; i < n; ++i) S2[i] = -xi * w2 * w2 * 0.5 * p1[i] * p1[i];
    return TBS_REF_OK;
}

/* ---- Harmonic sources 2..5, Eqs. 28b-28e (sum-frequency terms only, the
 * difference terms are dropped); xi of PAPER.md:117.
 *   S_h(r) = -xi (h omega1)^2 C_h(r),
 *   C_2 = psi1^2/2, C_3 = psi1 psi2, C_4 = psi2^2/2 + psi1 psi3, C_5 = psi2 psi3 + psi1 psi4.
 * psi_reim[m] is the field of harmonic m+1 (only those below h are read). */
int tbs_ref_harmonic_source(int64_t n, int h, const double *const *psi_reim, double beta, double rho0,
                            double c0, double f1_hz, double *S_reim) {
    if (n <= 0 || h < 2 || h > 5 || rho0 <= 0 || c0 <= 0) return TBS_REF_ERR_INVALID_ARG;
    const cplx *p1 = (const cplx *)psi_reim[0];
    const cplx *p2 = h >= 3 ? (const cplx *)psi_reim[1] : NULL;
    const cplx *p3 = h >= 4 ? (const cplx *)psi_reim[2] : NULL;
    const cplx *p4 = h >= 5 ? (const cplx *)psi_reim[3] : NULL;
    cplx *S = (cplx *)S_reim;
    double xi = beta / (rho0 * c0 * c0 * c0 * c0);
    double wh = (double)h * (2.0 * PI * f1_hz);
    for (int64_t i = 0; i < n; ++i) {
        cplx C;
        if (h == 2) C = 0.5 * p1[i] * p1[i];
        else if (h == 3) C = p1[i] * p2[i];
        else if (h == 4) C = 0.5 * p2[i] * p2[i] + p1[i] * p3[i];
        else C = p2[i] * p3[i] + p1[i] * p4[i];
        S[i] = -xi * wh * wh * C;
    }
    return TBS_REF_OK;
}
