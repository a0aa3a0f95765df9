// setup_kernels.cuh -- once-per-plan / once-per-medium kernels.
// All evaluate in double and store float, so the hot path sees correctly rounded inputs.
#pragma once
#include "fft_engine.cuh"

namespace tbs {

// Per-stage twiddle tables (fft_engine.cuh "Luts"), k-major [R][S], evaluated in double:
//   which = 0: lut[k][t] = exp(-2 pi i k t / L)            (L = N: table A;  L = S1: table C)
//   which = 1: lut[k][t] = exp(-2 pi i (2k+1) t / (2 L))   (L = N: table B)
// t < S = L / R, k < R.
__global__ void k_stage_lut(float2 *lut, int L, int R, int which) {
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    const int S = L / R;
    if (i >= S * R) return;
    const int k = i / S, t = i % S;
    double s, c;
    if (which == 0) sincospi(-2.0 * (double)((long long)k * t % L) / (double)L, &s, &c);
    else sincospi(-2.0 * (double)((long long)(2 * k + 1) * t % (2 * L)) / (double)(2 * L), &s, &c);
    lut[i] = make_float2((float)c, (float)s);
}

// First/last-stage tables A and B interleaved for the packed engine (fft_engine_x2.cuh):
// lut[k][t] = (A.x, B.x, A.y, B.y), A = exp(-2 pi i k t / N), B = exp(-2 pi i (2k+1) t / (2N)).
// same_lanes = 1 (periodic, unpadded form: both lanes are whole lines): B = A.
__global__ void k_stage_lut_ab(float4 *lut, int N, int R, int same_lanes) {
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    const int S = N / R;
    if (i >= S * R) return;
    const int k = i / S, t = i % S;
    double sa, ca, sb, cb;
    sincospi(-2.0 * (double)((long long)k * t % N) / (double)N, &sa, &ca);
    sincospi(-2.0 * (double)((long long)(2 * k + 1) * t % (2 * N)) / (double)(2 * N), &sb, &cb);
    if (same_lanes) { cb = ca; sb = sa; }
    lut[i] = make_float4((float)ca, (float)cb, (float)sa, (float)sb);
}

// Frequency index held at `pos` of a length-N DIF transform with radices r1, r2 (0 = none), rl.
__host__ __device__ inline int freq_of_pos(int pos, int N, int r1, int r2, int rl) {
    const int s1 = N / r1;
    const int k1 = pos / s1;
    int rem = pos % s1;
    if (r2 > 0) {
        const int s2 = s1 / r2;
        const int k2 = rem / s2;
        const int k3 = rem % s2;
        return k1 + r1 * (k2 + r2 * k3);
    }
    return k1 + r1 * rem;
}

// Green's-spectrum axis table (Alg. 1 l.9-10, in FFT order rather than centred +
// fftShift): p2[P] = (2 pi F~/(M dx))^2 / k0^2 for the padded-grid frequency F held at
// index P of a transformed line, F~ = F for F < M/2, F - M otherwise.
//   periodic = 1: see the last statement.
//   mult = 1, or k0^2/eps for the line-axis table of k_conv (fft_engine_x2.cuh, pmid_conv_item_pp).
//   xorder = 0 (k_col lines): P = s*N + pos, F = 2 freqN(pos) + s.
//   xorder = 1 (W rows of k_row; line-axis table of k_conv's fused middle stage):
//                P = 2 q + s, q = k*(N/rl) + b, pos = b*rl + k.
__global__ void k_axis_table(float *p2, int N, int r1, int r2, int rl, double dx, double k0, int xorder, double mult,
                             int periodic) {
    const int P = blockIdx.x * blockDim.x + threadIdx.x;
    const int M = 2 * N;
    if (P >= M) return;
    int s, pos;
    if (xorder) {
        const int q = P >> 1, nbl = N / rl;
        s = P & 1;
        pos = (q % nbl) * rl + q / nbl;
    } else {
        s = P / N;
        pos = P % N;
    }
    const int F = 2 * freq_of_pos(pos, N, r1, r2, rl) + s;
    const double Ft = (F < M / 2) ? (double)F : (double)(F - M);
    const double p = 2.0 * 3.14159265358979323846 * Ft / ((double)M * dx);
    // periodic boundary: only the even padded frequencies F = 2k exist (they are the frequencies of the
    // unpadded N-grid); an entry of 1e18 makes ghat vanish (to 1e-18) at the odd ones in every kernel
    // periodic = 2 (unpadded periodic kernels): entries 2q and 2q + 1 both hold the N-grid value of frequency q,
    // which is the padded grid's even frequency 2q
    if (periodic == 2) {
        const int Fe = F & ~1;
        const double Fte = (Fe < M / 2) ? (double)Fe : (double)(Fe - M);
        const double pe = 2.0 * 3.14159265358979323846 * Fte / ((double)M * dx);
        p2[P] = (float)((pe * pe) / (k0 * k0) * mult);
        return;
    }
    p2[P] = (periodic && s == 1) ? 1.0e18f : (float)((p * p) / (k0 * k0) * mult);
}

// Full Green's spectrum in natural FFT order, ghat = ((p2-k0^2) + i eps)/((p2-k0^2)^2 + eps^2)
// exactly as Alg. 1 l.12.  Tabulated form for inspection; the hot path recomputes
// ghat from the axis tables.
__global__ void k_green_spectrum(float2 *g, int mx, int my, int mz, double dx, double k0, double eps) {
    const long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    const long long tot = (long long)mx * my * mz;
    if (i >= tot) return;
    const int ix = (int)(i % mx), iy = (int)((i / mx) % my), iz = (int)(i / ((long long)mx * my));
    const double tp = 2.0 * 3.14159265358979323846;
    const double px = tp * (double)(ix < mx / 2 ? ix : ix - mx) / ((double)mx * dx);
    const double py = my > 1 ? tp * (double)(iy < my / 2 ? iy : iy - my) / ((double)my * dx) : 0.0;
    const double pz = mz > 1 ? tp * (double)(iz < mz / 2 ? iz : iz - mz) / ((double)mz * dx) : 0.0;
    const double a = px * px + py * py + pz * pz - k0 * k0;
    const double D = a * a + eps * eps;
    g[i] = make_float2((float)(a / D), (float)(eps / D));
}

// Medium -> non-dimensional potential V/k0^2 (absorption reading A6):
//   ktilde = w/c + alpha (tan(pi y/2) + i), alpha = alpha0_SI w^y, V = ktilde^2 - k0^2 - i eps.
__global__ void k_potential(float2 *V, const float *c, const float *alpha0_map, double alpha0_db,
                            double y, double omega, double k0, double damping, long long n) {
    const long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n) return;
    const double a0 = alpha0_map ? (double)alpha0_map[i] : alpha0_db;
    double kr = omega / (double)c[i], ki = 0.0;
    if (a0 != 0.0) {
        const double a0si = a0 * 100.0 / 8.685889638 / pow(2.0 * 3.14159265358979323846 * 1.0e6, y);
        const double alpha = a0si * pow(omega, y);
        kr += alpha * tan(3.14159265358979323846 * y / 2.0);
        ki = alpha;
    }
    const double k2 = k0 * k0;
    V[i] = make_float2((float)((kr * kr - ki * ki - k2) / k2), (float)((2.0 * kr * ki) / k2 - damping));
}

// Spatial part of the potential next to the k-space multiplier of Eq. 24: U_s/k0^2 = ((w/c)^2 - k0^2)/k0^2, real
// (Eq. 25 without the -i eps, which the multiplier carries).
__global__ void k_scatterer_potential(float2 *V, const float *c, double omega, double k0, long long n) {
    const long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n) return;
    const double kr = omega / (double)c[i];
    V[i] = make_float2((float)((kr * kr - k0 * k0) / (k0 * k0)), 0.f);
}

// Raw V (1/m^2) -> V/k0^2
__global__ void k_scale_complex(float2 *dst, const float2 *src, double s, long long n) {
    const long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n) return;
    dst[i] = make_float2((float)((double)src[i].x * s), (float)((double)src[i].y * s));
}

// Source deposition with multilinear weights (reading A9; a node-aligned point is the paper's
// single-pixel source).  One thread per (source, corner).
__global__ void k_deposit(float2 *S, const double *pos, const float2 *amp, int n_src, int ndim,
                          int nx, int ny, int nz, double dx) {
    const int corners = 1 << ndim;
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n_src * corners) return;
    const int j = i / corners, cidx = i % corners;
    const int dims[3] = {nx, ny, nz};
    long long idx = 0, stride = 1;
    double w = 1.0;
    for (int a = 0; a < ndim; ++a) {
        const double g = pos[(long long)j * ndim + a] / dx;
        double fl = floor(g);
        if (fl > (double)(dims[a] - 2)) fl = (double)(dims[a] - 2);
        const double fr = g - fl;
        const int bit = (cidx >> a) & 1;
        w *= bit ? fr : 1.0 - fr;
        idx += ((long long)fl + bit) * stride;
        stride *= dims[a];
    }
    if (w == 0.0) return;
    atomicAdd(&S[idx].x, (float)((double)amp[j].x * w));
    atomicAdd(&S[idx].y, (float)((double)amp[j].y * w));
}

// Absorbing-layer window along one axis, Eq. 29, reading A4.
__global__ void k_abl_window(float *a, int n, int cells, double zeta_half_mu) {
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n) return;
    const int x = i < n - 1 - i ? i : n - 1 - i;
    double v = 1.0;
    if (cells > 0 && x < cells) {
        const double zeta = 2.0 * zeta_half_mu / (double)cells;
        v = 1.0 / (1.0 + exp(-zeta * ((double)x - 0.5 * (double)cells)));
    }
    a[i] = (float)v;
}

// max |p|^2 over one row (2-D) / plane (3-D), as the bit pattern of a non-negative float.
__global__ void k_row_max(const float2 *p, long long first, long long count, unsigned int *out) {
    const long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    float m = 0.f;
    if (i < count) {
        const float2 v = p[first + i];
        m = v.x * v.x + v.y * v.y;
    }
    for (int o = 16; o > 0; o >>= 1) m = fmaxf(m, __shfl_xor_sync(0xffffffffu, m, o));
    if ((threadIdx.x & 31) == 0) atomicMax(out, __float_as_uint(m));
}

// p1 <- g p1 with g = target / max|p1| over the reference row ("surface pressure", reading A10).
__global__ void k_rescale_field(float2 *p1, const unsigned int *max2bits, double target, long long n) {
    const long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n) return;
    const double g = target / sqrt((double)__uint_as_float(*max2bits));
    p1[i] = make_float2((float)((double)p1[i].x * g), (float)((double)p1[i].y * g));
}

// Harmonic source (Eqs. 28b-28e; xi = beta/(rho0 c0^4)):
//   S = coef (wab pa pb + wcd pc pd),  coef = -xi (h w1)^2;
//   h = 2: pa = pb = psi1, wab = 1/2;   h = 3: psi1 psi2;
//   h = 4: psi2 psi2 / 2 + psi1 psi3;   h = 5: psi2 psi3 + psi1 psi4   (pc = nullptr: one product).
__global__ void k_harmonic_source(float2 *S, double coef, const float2 *pa, const float2 *pb, double wab,
                                  const float2 *pc, const float2 *pd, double wcd, long long n) {
    const long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n) return;
    const double ar = pa[i].x, ai = pa[i].y, br = pb[i].x, bi = pb[i].y;
    double re = wab * (ar * br - ai * bi), im = wab * (ar * bi + ai * br);
    if (pc) {
        const double cr = pc[i].x, ci = pc[i].y, dr = pd[i].x, di = pd[i].y;
        re += wcd * (cr * dr - ci * di);
        im += wcd * (cr * di + ci * dr);
    }
    S[i] = make_float2((float)(coef * re), (float)(coef * im));
}

}  // namespace tbs
