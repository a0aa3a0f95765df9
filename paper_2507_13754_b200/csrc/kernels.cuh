// kernels.cuh -- the Born-term kernels, built on fft_engine.cuh.
//
//   k_row  (K1 / K3+K1 fused, "K31"): per grid row along x.
//          inverse half:  W row (2N positions) -> IFFT_x -> crop -> u = A.(.) -> p (+)= u,
//                         partial ||u||^2, ||p||^2 -> last CTA finalises r_n and the stop flag
//          forward half:  w = V.u (or the source S for term 0) -> zero-pad -> FFT_x -> W row
//          u never leaves the chip between the two halves (cross-term fusion).
//   k_col<MODE>: per tile of T adjacent lines along a strided axis (y in 2-D; y and z in 3-D).
//          CONV: pad, FFT, .ghat, IFFT, crop, in place   (K2 in 2-D, the z pass in 3-D)
//          FWD : pad, FFT  N -> 2N positions             (3-D y pass, forward)
//          INV : IFFT, crop  2N positions -> N           (3-D y pass, inverse)
#pragma once
#include "fft_engine.cuh"

namespace tbs {

// Device-resident loop control, one per frequency slot.
struct Ctl {
    int term;        // index of the next term to be added by k_row (0 = u_0)
    int done;        // set when the series stops; every kernel exits at once when it is set
    int status;      // tbs_status at the stop
    int max_terms;
    double tol;
    unsigned int ticket;  // CTAs of the current k_row launch that have finished
    int n_terms;     // index of the last term added
};

enum { MODE_CONV = 0, MODE_FWD = 1, MODE_INV = 2 };

struct ColArgs {
    const float2 *in;
    float2 *out;
    long long in_line_stride, out_line_stride;    // between consecutive positions of a line
    long long in_outer_stride, out_outer_stride;  // between consecutive outer indices
    int inner_len;                                // number of adjacent lines (multiple of T)
    const float *p2_line;   // [2N] |p|^2/k0^2 of this axis, position order       (CONV)
    const float *p2_inner;  // [inner_len] of the inner (x) axis, position order  (CONV)
    const float *p2_outer;  // [n_outer] of the outer axis or nullptr             (CONV)
    float e, scale;         // eps/k0^2 and 1/prod(2N)                            (CONV)
    const float2 *tw;
    const Ctl *ctl;
};

template <int N, int T, int NT, int MODE>
__global__ void __launch_bounds__(NT) k_col(ColArgs a) {
    using P = Radix<N>;
    constexpr int R1 = P::R1, R2 = P::R2, RL = P::RL;
    constexpr int S1 = N / R1;
    static_assert((S1 * T) % NT == 0 && NT % T == 0, "tile/thread mismatch");
    constexpr int NB = (S1 * T) / NT;  // first/last-stage butterflies per thread
    constexpr int TSTEP = NT / T;
    constexpr int M = 2 * N;
    using Lay = ColLay<N, T, RL>;
    extern __shared__ float2 sm[];
    if (a.ctl->done) return;

    const int tid = threadIdx.x;
    const int line = tid % T, t0 = tid / T;
    const int tiles = a.inner_len / T;
    const int inner0 = (blockIdx.x % tiles) * T;
    const int outer = blockIdx.x / tiles;
    const float2 *in = a.in + (long long)outer * a.in_outer_stride + inner0 + line;
    float2 *out = a.out + (long long)outer * a.out_outer_stride + inner0 + line;
    const float2 *__restrict__ tw = a.tw;

    float a_line = 0.f;
    if (MODE == MODE_CONV) {
        a_line = __ldg(&a.p2_inner[inner0 + line]) - 1.0f;
        if (a.p2_outer) a_line += __ldg(&a.p2_outer[outer]);
    }

    float2 acc[NB][R1];
#pragma unroll
    for (int s = 0; s < 2; ++s) {
        // ---- forward half: N inputs (twisted for s = 1) -> smem, or (INV) load positions ----
        if (MODE != MODE_INV) {
#pragma unroll
            for (int i = 0; i < NB; ++i) {
                const int t = t0 + i * TSTEP;
                float2 x[R1];
#pragma unroll
                for (int j = 0; j < R1; ++j) {
                    const int pos = t + j * S1;
                    float2 v = in[(long long)pos * a.in_line_stride];
                    if (s) v = cmul(v, __ldg(&tw[pos * (NTW / M)]));
                    x[j] = v;
                }
                first_fwd<N, R1, Lay>(x, line, t, sm, tw);
            }
            __syncthreads();
            if (R2 > 0) {
                stage_smem<N, S1, (R2 > 0 ? R2 : 2), true, Lay, NT>(sm, tw, tid, (N / (R2 > 0 ? R2 : 2)) * T);
                __syncthreads();
            }
        }
        if (MODE == MODE_CONV) {
            mid_conv<N, RL, Lay, NT>(sm, tid, (N / RL) * T, a.p2_line + s * N, a_line, a.e, a.scale);
            __syncthreads();
        } else if (MODE == MODE_FWD) {
            // last forward stage straight to global: positions s*N + b*RL + k
            for (int w = tid; w < (N / RL) * T; w += NT) {
                const int b = w / T;
                float2 v[RL];
#pragma unroll
                for (int j = 0; j < RL; ++j) v[j] = sm[Lay::addr(line, b * RL + j)];
                bfly<RL, -1>(v);
#pragma unroll
                for (int i = 0; i < RL; ++i)
                    out[(long long)(s * N + b * RL + brev(i, RL)) * a.out_line_stride] = v[i];
            }
            __syncthreads();
        } else {
            // INV: first inverse stage straight from global
            for (int w = tid; w < (N / RL) * T; w += NT) {
                const int b = w / T;
                float2 v[RL];
#pragma unroll
                for (int k = 0; k < RL; ++k) v[k] = in[(long long)(s * N + b * RL + k) * a.in_line_stride];
                bfly<RL, +1>(v);
#pragma unroll
                for (int i = 0; i < RL; ++i) sm[Lay::addr(line, b * RL + brev(i, RL))] = v[i];
            }
            __syncthreads();
        }
        // ---- inverse half ----
        if (MODE != MODE_FWD) {
            if (R2 > 0) {
                stage_smem<N, S1, (R2 > 0 ? R2 : 2), false, Lay, NT>(sm, tw, tid, (N / (R2 > 0 ? R2 : 2)) * T);
                __syncthreads();
            }
#pragma unroll
            for (int i = 0; i < NB; ++i) {
                const int t = t0 + i * TSTEP;
                float2 z[R1];
                last_inv<N, R1, Lay>(z, line, t, sm, tw);
#pragma unroll
                for (int j = 0; j < R1; ++j) {
                    if (s == 0) acc[i][j] = z[j];
                    else acc[i][j] = cadd(acc[i][j], cmulc(z[j], __ldg(&tw[(t + j * S1) * (NTW / M)])));
                }
            }
            __syncthreads();
        }
    }
    if (MODE != MODE_FWD) {
#pragma unroll
        for (int i = 0; i < NB; ++i) {
            const int t = t0 + i * TSTEP;
#pragma unroll
            for (int j = 0; j < R1; ++j) {
                float2 v = acc[i][j];
                if (MODE == MODE_INV) { v.x *= a.scale; v.y *= a.scale; }
                out[(long long)(t + j * S1) * a.out_line_stride] = v;
            }
        }
    }
}

struct RowArgs {
    float2 *W;            // [rows][2N] intermediate, position order along x, updated in place
    const float2 *src;    // FIRST: source / input field [rows][N]
    const float2 *V;      // [rows][N] non-dimensional potential V/k0^2
    float2 *p;            // [rows][N] running field
    const float *ax;      // [N] ABL window along x
    const float *ay;      // [ny] ABL window along y
    const float *az;      // [nz] or nullptr
    int ny;               // rows = ny * nz; row = z*ny + y
    int rows;
    float src_scale;      // FIRST: 1/k0^2
    int do_fwd;           // 0: stop after the inverse half (tbs_apply_green)
    double *norms;        // [max_terms+1][2] sum |u|^2, sum |p|^2
    double *history;      // [max_terms+1]
    Ctl *ctl;
    const float2 *tw;
};

// FIRST = true : forward half only, w = src * src_scale (term 0: u_0 = G S, Eq. 20)
// FIRST = false: inverse half (K3) + forward half (K1) of the next term
template <int N, int ROWS, int NT, bool FIRST>
__global__ void __launch_bounds__(NT) k_row(RowArgs a) {
    using P = Radix<N>;
    constexpr int R1 = P::R1, R2 = P::R2, RL = P::RL;
    constexpr int S1 = N / R1;
    static_assert((ROWS * S1) % NT == 0, "tile/thread mismatch");
    constexpr int NB = (ROWS * S1) / NT;
    constexpr int M = 2 * N;
    using Lay = RowLay<N>;
    extern __shared__ float2 sm[];
    __shared__ float red[2][32];
    if (a.ctl->done) return;

    const int tid = threadIdx.x;
    const int row0 = blockIdx.x * ROWS;
    const float2 *__restrict__ tw = a.tw;
    float2 x[NB][R1];
    const int term = FIRST ? 0 : a.ctl->term;

    if (!FIRST) {
        // ---------------- inverse half: IFFT_x, crop, window, accumulate ----------------
#pragma unroll
        for (int s = 0; s < 2; ++s) {
            for (int e = tid; e < ROWS * N; e += NT) {
                const int l = e / N, pos = e % N;
                sm[Lay::addr(l, pos)] = a.W[(long long)(row0 + l) * M + s * N + pos];
            }
            __syncthreads();
            stage_smem<N, RL, RL, false, Lay, NT>(sm, tw, tid, ROWS * (N / RL));
            __syncthreads();
            if (R2 > 0) {
                stage_smem<N, S1, (R2 > 0 ? R2 : 2), false, Lay, NT>(sm, tw, tid, ROWS * (N / (R2 > 0 ? R2 : 2)));
                __syncthreads();
            }
#pragma unroll
            for (int i = 0; i < NB; ++i) {
                const int w = tid + i * NT;
                const int t = w % S1, l = w / S1;
                float2 z[R1];
                last_inv<N, R1, Lay>(z, l, t, sm, tw);
#pragma unroll
                for (int j = 0; j < R1; ++j) {
                    if (s == 0) x[i][j] = z[j];
                    else x[i][j] = cadd(x[i][j], cmulc(z[j], __ldg(&tw[(t + j * S1) * (NTW / M)])));
                }
            }
            __syncthreads();
        }
        // u = A . crop(...);  p (+)= u;  norms;  w = V . u
        float uu = 0.f, pp = 0.f;
#pragma unroll
        for (int i = 0; i < NB; ++i) {
            const int w = tid + i * NT;
            const int t = w % S1, l = w / S1;
            const int row = row0 + l;
            float wrow = __ldg(&a.ay[row % a.ny]);
            if (a.az) wrow *= __ldg(&a.az[row / a.ny]);
#pragma unroll
            for (int j = 0; j < R1; ++j) {
                const int pos = t + j * S1;
                const long long gi = (long long)row * N + pos;
                const float wgt = wrow * __ldg(&a.ax[pos]);
                float2 u = make_float2(x[i][j].x * wgt, x[i][j].y * wgt);
                float2 pv = u;
                if (term > 0) pv = cadd(a.p[gi], u);
                a.p[gi] = pv;
                uu = fmaf(u.x, u.x, fmaf(u.y, u.y, uu));
                pp = fmaf(pv.x, pv.x, fmaf(pv.y, pv.y, pp));
                x[i][j] = cmul(__ldg(&a.V[gi]), u);
            }
        }
        // block reduction (warp shuffles, then one double atomic per CTA and quantity)
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) {
            uu += __shfl_xor_sync(0xffffffffu, uu, o);
            pp += __shfl_xor_sync(0xffffffffu, pp, o);
        }
        if ((tid & 31) == 0) { red[0][tid >> 5] = uu; red[1][tid >> 5] = pp; }
        __syncthreads();
        if (tid == 0) {
            double su = 0.0, sp = 0.0;
            for (int w = 0; w < NT / 32; ++w) { su += (double)red[0][w]; sp += (double)red[1][w]; }
            atomicAdd(&a.norms[2 * term], su);
            atomicAdd(&a.norms[2 * term + 1], sp);
            __threadfence();
            const unsigned int tk = atomicAdd(&a.ctl->ticket, 1u);
            if (tk == gridDim.x - 1) {
                // last CTA of this launch: finalise the term
                __threadfence();
                const double nu = *((volatile double *)&a.norms[2 * term]);
                const double np = *((volatile double *)&a.norms[2 * term + 1]);
                const double r = sqrt(nu) / sqrt(np);
                a.history[term] = (term == 0) ? 1.0 : r;
                a.ctl->ticket = 0;
                a.ctl->n_terms = term;
                a.ctl->term = term + 1;
                if (!(r == r) || r > 1.0e300 || !(np > 0.0 || nu == 0.0)) {
                    if (!(nu == 0.0 && np == 0.0)) { a.ctl->done = 1; a.ctl->status = -5; }
                    else { a.ctl->done = 1; a.ctl->status = 0; }
                } else if (term >= 1 && r < a.ctl->tol) {
                    a.ctl->done = 1; a.ctl->status = 0;
                } else if (term >= a.ctl->max_terms) {
                    a.ctl->done = 1; a.ctl->status = 1;
                }
            }
        }
        if (!a.do_fwd) return;
    } else {
#pragma unroll
        for (int i = 0; i < NB; ++i) {
            const int w = tid + i * NT;
            const int t = w % S1, l = w / S1;
#pragma unroll
            for (int j = 0; j < R1; ++j) {
                float2 v = a.src[(long long)(row0 + l) * N + t + j * S1];
                x[i][j] = make_float2(v.x * a.src_scale, v.y * a.src_scale);
            }
        }
    }

    // ---------------- forward half: zero-pad (two parity halves), FFT_x ----------------
#pragma unroll
    for (int s = 0; s < 2; ++s) {
#pragma unroll
        for (int i = 0; i < NB; ++i) {
            const int w = tid + i * NT;
            const int t = w % S1, l = w / S1;
            float2 y[R1];
#pragma unroll
            for (int j = 0; j < R1; ++j) {
                y[j] = x[i][j];
                if (s) y[j] = cmul(y[j], __ldg(&tw[(t + j * S1) * (NTW / M)]));
            }
            first_fwd<N, R1, Lay>(y, l, t, sm, tw);
        }
        __syncthreads();
        if (R2 > 0) {
            stage_smem<N, S1, (R2 > 0 ? R2 : 2), true, Lay, NT>(sm, tw, tid, ROWS * (N / (R2 > 0 ? R2 : 2)));
            __syncthreads();
        }
        stage_smem<N, RL, RL, true, Lay, NT>(sm, tw, tid, ROWS * (N / RL));
        __syncthreads();
        for (int e = tid; e < ROWS * N; e += NT) {
            const int l = e / N, pos = e % N;
            a.W[(long long)(row0 + l) * M + s * N + pos] = sm[Lay::addr(l, pos)];
        }
        __syncthreads();
    }
}

}  // namespace tbs
