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
// Both parity halves of a padded line (fft_engine.cuh) are resident in shared memory at once, so
// the input is read once and the twiddles of a butterfly pair are fetched once.
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
    Luts lut;
    const Ctl *ctl;
};

template <int N, int T, int NT, int MODE>
__global__ void __launch_bounds__(NT) k_col(ColArgs a) {
    using P = Radix<N>;
    constexpr int R1 = P::R1, R2 = P::R2, RL = P::RL;
    constexpr int R2s = R2 > 0 ? R2 : 2;
    constexpr int S1 = N / R1;
    static_assert((S1 * T) % NT == 0 && NT % T == 0, "tile/thread mismatch");
    constexpr int NB = (S1 * T) / NT;  // first/last-stage butterfly pairs per thread
    constexpr int TSTEP = NT / T;
    constexpr int HALF = N * T;
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

    // ---- forward: N inputs -> both halves in smem ----
    if (MODE != MODE_INV) {
#pragma unroll
        for (int i = 0; i < NB; ++i) {
            const int t = t0 + i * TSTEP;
            float2 x[R1];
#pragma unroll
            for (int j = 0; j < R1; ++j) x[j] = in[(long long)(t + j * S1) * a.in_line_stride];
            first_fwd_pair<N, R1, Lay, HALF>(x, line, t, sm, a.lut);
        }
        __syncthreads();
        if (R2 > 0) {
            stage_pair<N, S1, R2s, true, Lay, NT, HALF>(sm, a.lut.C, tid, (N / R2s) * T);
            __syncthreads();
        }
    }
    if (MODE == MODE_CONV) {
        float a_line = __ldg(&a.p2_inner[inner0 + line]) - 1.0f;
        if (a.p2_outer) a_line += __ldg(&a.p2_outer[outer]);
        mid_conv_pair<N, RL, Lay, NT, HALF>(sm, tid, (N / RL) * T, a.p2_line, a_line, a.e, a.scale);
        __syncthreads();
    } else if (MODE == MODE_FWD) {
        // last forward stage straight to global: positions s*N + b*RL + k
        for (int w = tid; w < (N / RL) * T; w += NT) {
            const int b = w / T;
#pragma unroll
            for (int s = 0; s < 2; ++s) {
                float2 v[RL];
#pragma unroll
                for (int j = 0; j < RL; ++j) v[j] = sm[s * HALF + Lay::addr(line, b * RL + j)];
                bfly<RL, -1>(v);
#pragma unroll
                for (int i = 0; i < RL; ++i)
                    out[(long long)(s * N + b * RL + brev(i, RL)) * a.out_line_stride] = v[i];
            }
        }
        return;
    } else {
        // INV: first inverse stage straight from global
        for (int w = tid; w < (N / RL) * T; w += NT) {
            const int b = w / T;
#pragma unroll
            for (int s = 0; s < 2; ++s) {
                float2 v[RL];
#pragma unroll
                for (int k = 0; k < RL; ++k) v[k] = in[(long long)(s * N + b * RL + k) * a.in_line_stride];
                bfly<RL, +1>(v);
#pragma unroll
                for (int i = 0; i < RL; ++i) sm[s * HALF + Lay::addr(line, b * RL + brev(i, RL))] = v[i];
            }
        }
        __syncthreads();
    }
    // ---- inverse: both halves -> N outputs ----
    if (R2 > 0) {
        stage_pair<N, S1, R2s, false, Lay, NT, HALF>(sm, a.lut.C, tid, (N / R2s) * T);
        __syncthreads();
    }
#pragma unroll
    for (int i = 0; i < NB; ++i) {
        const int t = t0 + i * TSTEP;
        float2 z[R1];
        last_inv_pair<N, R1, Lay, HALF>(z, line, t, sm, a.lut);
#pragma unroll
        for (int j = 0; j < R1; ++j) out[(long long)(t + j * S1) * a.out_line_stride] = z[j];
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
    Luts lut;
};

// RL contiguous complex values <-> registers with 128-bit accesses (RL*8 bytes, 16-byte aligned).
template <int RL>
__device__ __forceinline__ void load_chunk(float2 (&v)[RL], const float2 *g) {
    const float4 *p = reinterpret_cast<const float4 *>(g);
#pragma unroll
    for (int q = 0; q < RL / 2; ++q) {
        const float4 f = p[q];
        v[2 * q] = make_float2(f.x, f.y);
        v[2 * q + 1] = make_float2(f.z, f.w);
    }
}

// FIRST = true : forward half only, w = src * src_scale (term 0: u_0 = G S, Eq. 20)
// FIRST = false: inverse half (K3) + forward half (K1) of the next term
template <int N, int ROWS, int NT, int MINB, bool FIRST>
__global__ void __launch_bounds__(NT, MINB) k_row(RowArgs a) {
    using P = Radix<N>;
    constexpr int R1 = P::R1, R2 = P::R2, RL = P::RL;
    constexpr int R2s = R2 > 0 ? R2 : 2;
    constexpr int S1 = N / R1;
    static_assert((ROWS * S1) % NT == 0, "tile/thread mismatch");
    constexpr int NB = (ROWS * S1) / NT;
    constexpr int M = 2 * N;
    using Lay = RowLay<N>;
    constexpr int HALF = ROWS * Lay::PITCH;
    extern __shared__ float2 sm[];
    __shared__ float red[2][32];
    if (a.ctl->done) return;

    const int tid = threadIdx.x;
    const int row0 = blockIdx.x * ROWS;
    float2 x[NB][R1];
    const int term = FIRST ? 0 : a.ctl->term;

    if (!FIRST) {
        // ---------------- inverse half: IFFT_x, crop, window, accumulate ----------------
        // first inverse stage (contiguous blocks of RL) straight from global memory
        for (int w = tid; w < ROWS * (N / RL); w += NT) {
            const int b = w % (N / RL), l = w / (N / RL);
#pragma unroll
            for (int s = 0; s < 2; ++s) {
                float2 v[RL];
                load_chunk<RL>(v, a.W + (long long)(row0 + l) * M + s * N + b * RL);
                bfly<RL, +1>(v);
#pragma unroll
                for (int i = 0; i < RL; ++i) sm[s * HALF + Lay::addr(l, b * RL + brev(i, RL))] = v[i];
            }
        }
        __syncthreads();
        if (R2 > 0) {
            stage_pair<N, S1, R2s, false, Lay, NT, HALF>(sm, a.lut.C, tid, ROWS * (N / R2s));
            __syncthreads();
        }
        // last inverse stage + crop + window + accumulate; the same thread later writes the same
        // smem slots in the forward half, so no barrier is needed in between
        float uu = 0.f, pp = 0.f;
#pragma unroll
        for (int i = 0; i < NB; ++i) {
            const int w = tid + i * NT;
            const int t = w % S1, l = w / S1;
            last_inv_pair<N, R1, Lay, HALF>(x[i], l, t, sm, a.lut);
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
                if (!(r == r) || r > 1.0e300) {
                    a.ctl->done = 1; a.ctl->status = -5;
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
    for (int i = 0; i < NB; ++i) {
        const int w = tid + i * NT;
        const int t = w % S1, l = w / S1;
        first_fwd_pair<N, R1, Lay, HALF>(x[i], l, t, sm, a.lut);
    }
    __syncthreads();
    if (R2 > 0) {
        stage_pair<N, S1, R2s, true, Lay, NT, HALF>(sm, a.lut.C, tid, ROWS * (N / R2s));
        __syncthreads();
    }
    // last forward stage (contiguous blocks of RL) straight to global memory
    for (int w = tid; w < ROWS * (N / RL); w += NT) {
        const int b = w % (N / RL), l = w / (N / RL);
#pragma unroll
        for (int s = 0; s < 2; ++s) {
            float2 v[RL];
#pragma unroll
            for (int j = 0; j < RL; ++j) v[j] = sm[s * HALF + Lay::addr(l, b * RL + j)];
            bfly<RL, -1>(v);
            // v[i] = X[brev(i)]: gather into natural order and store 2 values per 128-bit write
            float2 o[RL];
#pragma unroll
            for (int i = 0; i < RL; ++i) o[brev(i, RL)] = v[i];
            float4 *g = reinterpret_cast<float4 *>(a.W + (long long)(row0 + l) * M + s * N + b * RL);
#pragma unroll
            for (int q = 0; q < RL / 2; ++q) g[q] = make_float4(o[2 * q].x, o[2 * q].y, o[2 * q + 1].x, o[2 * q + 1].y);
        }
    }
}

}  // namespace tbs
