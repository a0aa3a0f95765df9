// fft_engine_x2.cuh -- the packed ("x2") form of the shared-memory FFT stages (sm_100a f32x2 pipe).
//
// The two parity halves of a zero-padded line (fft_engine.cuh: X[2k+s], s = 0, 1) go through the
// same butterflies with the same twiddles at every stage, so they are carried as ONE value
//   P2 = { re = (re_even, re_odd), im = (im_even, im_odd) }
// and every add / multiply is a packed FADD2 / FMUL2 / FFMA2: half the issue slots of the scalar
// form for the same FP32 results (the FP32 pipe itself is not wider: 128 results/clk/SM either way,
// measured), and half the shared-memory instructions (one 16-byte access per position).  A scalar
// twiddle is a broadcast operand and a negation an operand modifier, so no extra moves are issued.
// Shared-memory element: float4 (re_even, re_odd, im_even, im_odd) per position.
#pragma once
#include "fft_engine.cuh"

namespace tbs {

struct P2 {
    float2 re, im;
};

__device__ __forceinline__ float2 f2(float a) { return make_float2(a, a); }
__device__ __forceinline__ float2 neg2(float2 a) { return make_float2(-a.x, -a.y); }
__device__ __forceinline__ P2 padd(P2 a, P2 b) { return P2{__fadd2_rn(a.re, b.re), __fadd2_rn(a.im, b.im)}; }
__device__ __forceinline__ P2 psub(P2 a, P2 b) { return P2{__fadd2_rn(a.re, neg2(b.re)), __fadd2_rn(a.im, neg2(b.im))}; }
// a * w, w a scalar complex (broadcast to both halves)
__device__ __forceinline__ P2 pmul(P2 a, float2 w) {
    return P2{__ffma2_rn(a.re, f2(w.x), __fmul2_rn(a.im, f2(-w.y))), __ffma2_rn(a.re, f2(w.y), __fmul2_rn(a.im, f2(w.x)))};
}
// a * conj(w)
__device__ __forceinline__ P2 pmulc(P2 a, float2 w) {
    return P2{__ffma2_rn(a.re, f2(w.x), __fmul2_rn(a.im, f2(w.y))), __ffma2_rn(a.im, f2(w.x), __fmul2_rn(a.re, f2(-w.y)))};
}
// a * w, w = (wre, wim) a different twiddle per half
__device__ __forceinline__ P2 pmul2(P2 a, float2 wre, float2 wim) {
    return P2{__ffma2_rn(a.re, wre, __fmul2_rn(a.im, neg2(wim))), __ffma2_rn(a.re, wim, __fmul2_rn(a.im, wre))};
}
__device__ __forceinline__ P2 pmulc2(P2 a, float2 wre, float2 wim) {
    return P2{__ffma2_rn(a.re, wre, __fmul2_rn(a.im, wim)), __ffma2_rn(a.im, wre, __fmul2_rn(a.re, neg2(wim)))};
}

// d * w_16^(idx16) with sign SGN, both halves (packed form of mul_w16).
template <int SGN>
__device__ __forceinline__ P2 pmul_w16(P2 d, int idx16) {
    constexpr float C1 = 0.92387953251128674f;  // cos(pi/8)
    constexpr float S1 = 0.38268343236508977f;  // sin(pi/8)
    constexpr float H = 0.70710678118654752f;   // sqrt(1/2)
    constexpr float s = (float)SGN;
    switch (idx16) {
        case 0: return d;
        case 1: return pmul(d, make_float2(C1, s * S1));
        case 2: return P2{__fmul2_rn(__fadd2_rn(d.re, SGN > 0 ? neg2(d.im) : d.im), f2(H)),
                          __fmul2_rn(__fadd2_rn(d.im, SGN > 0 ? d.re : neg2(d.re)), f2(H))};
        case 3: return pmul(d, make_float2(S1, s * C1));
        case 4: return SGN > 0 ? P2{neg2(d.im), d.re} : P2{d.im, neg2(d.re)};
        case 5: return pmul(d, make_float2(-S1, s * C1));
        case 6: return P2{__fmul2_rn(__fadd2_rn(neg2(d.re), SGN > 0 ? neg2(d.im) : d.im), f2(H)),
                          __fmul2_rn(__fadd2_rn(neg2(d.im), SGN > 0 ? d.re : neg2(d.re)), f2(H))};
        default: return pmul(d, make_float2(-C1, s * S1));
    }
}

// w_16^idx = (w16x, SGN * w16y), idx = 0..7.
__device__ __forceinline__ constexpr float w16x(int idx) {
    constexpr float C1 = 0.92387953251128674f, S1 = 0.38268343236508977f, H = 0.70710678118654752f;
    return idx == 0 ? 1.f : idx == 1 ? C1 : idx == 2 ? H : idx == 3 ? S1 : idx == 4 ? 0.f : idx == 5 ? -S1 : idx == 6 ? -H : -C1;
}
__device__ __forceinline__ constexpr float w16y(int idx) {
    constexpr float C1 = 0.92387953251128674f, S1 = 0.38268343236508977f, H = 0.70710678118654752f;
    return idx == 0 ? 0.f : idx == 1 ? S1 : idx == 2 ? H : idx == 3 ? C1 : idx == 4 ? 1.f : idx == 5 ? C1 : idx == 6 ? H : S1;
}

// Butterfly with the twiddle of its second operand folded in: s = a + b w, d = a - b w = 2a - s.
// b w is never formed: 6 packed operations instead of 4 (multiply) + 4 (add, subtract).
__device__ __forceinline__ void pbfly_tw(P2 a, P2 b, float2 wre, float2 wim, P2 &s, P2 &d) {
    s.re = __ffma2_rn(b.re, wre, __ffma2_rn(b.im, neg2(wim), a.re));
    s.im = __ffma2_rn(b.re, wim, __ffma2_rn(b.im, wre, a.im));
    d.re = __ffma2_rn(a.re, f2(2.0f), neg2(s.re));
    d.im = __ffma2_rn(a.im, f2(2.0f), neg2(s.im));
}

// Radix-2 layers h = H0 .. 1 of the DFT_R butterfly.  pend[i] is the power of w_16 that v[i] still has
// to be multiplied by (all indices are compile-time constants after unrolling): a factor owed by the
// first operand of a butterfly is applied there, one owed by the second operand goes into pbfly_tw.
template <int R, int SGN, int H0>
__device__ __forceinline__ void pbfly_layers(P2 (&v)[R], int (&pend)[R]) {
#pragma unroll
    for (int h = H0; h >= 1; h >>= 1) {
#pragma unroll
        for (int g = 0; g < R; g += 2 * h) {
#pragma unroll
            for (int m = 0; m < h; ++m) {
                const int ia = g + m, ib = g + m + h;
                const P2 a = pmul_w16<SGN>(v[ia], pend[ia]);
                const int pb = pend[ib];
                if (pb == 0 || pb == 4) {
                    const P2 b = pmul_w16<SGN>(v[ib], pb);
                    v[ia] = padd(a, b);
                    v[ib] = psub(a, b);
                } else {
                    pbfly_tw(a, v[ib], f2(w16x(pb)), f2((float)SGN * w16y(pb)), v[ia], v[ib]);
                }
                pend[ia] = 0;
                pend[ib] = m * (8 / h);
            }
        }
    }
}

// DFT_R of v (sign SGN), natural order in, BIT-REVERSED order out, both halves at once.
template <int R, int SGN>
__device__ __forceinline__ void pbfly(P2 (&v)[R]) {
    int pend[R];
#pragma unroll
    for (int i = 0; i < R; ++i) pend[i] = 0;
    pbfly_layers<R, SGN, R / 2>(v, pend);
}

// Inverse (DIT) butterfly with its input twiddles: DFT_R(+1) of v[k] conj(w[k]), w[k] = (wre[k], wim[k])
// per half (w[0] too: the odd half carries the padding twist).  The twiddles of the upper half go into
// the first layer.
template <int R>
__device__ __forceinline__ void pbfly_dit(P2 (&v)[R], const float2 (&wre)[R], const float2 (&wim)[R]) {
    constexpr int h = R / 2;
    int pend[R];
#pragma unroll
    for (int m = 0; m < h; ++m) {
        const P2 a = pmulc2(v[m], wre[m], wim[m]);
        pbfly_tw(a, v[m + h], wre[m + h], neg2(wim[m + h]), v[m], v[m + h]);
        pend[m] = 0;
        pend[m + h] = m * (8 / h);
    }
    pbfly_layers<R, +1, R / 4>(v, pend);
}
// the same with one scalar twiddle per position (both halves); w[0] = 1 is not applied
template <int R>
__device__ __forceinline__ void pbfly_dit(P2 (&v)[R], const float2 (&tw)[R]) {
    constexpr int h = R / 2;
    int pend[R];
#pragma unroll
    for (int m = 0; m < h; ++m) {
        const P2 a = m > 0 ? pmulc(v[m], tw[m]) : v[0];
        pbfly_tw(a, v[m + h], f2(tw[m + h].x), f2(-tw[m + h].y), v[m], v[m + h]);
        pend[m] = 0;
        pend[m + h] = m * (8 / h);
    }
    pbfly_layers<R, +1, R / 4>(v, pend);
}

__device__ __forceinline__ P2 lds_p2(const float4 *p) {
    const float4 f = *p;
    return P2{make_float2(f.x, f.y), make_float2(f.z, f.w)};
}
__device__ __forceinline__ void sts_p2(float4 *p, P2 v) { *p = make_float4(v.re.x, v.re.y, v.im.x, v.im.y); }

// Packed line layout: one float4 (16-byte slot) per position, N slots per line, no padding.  The slot
// index is the position with bits 4-6 XORed into bits 0-2: every access pattern of the stages (threads
// on consecutive positions; threads on consecutive blocks of 16 reading the same offset; strides of 16
// inside a block of 256) then touches 8 different 16-byte banks per quarter-warp.
template <int N>
struct LineLay {
    static constexpr int PITCH = N;
    __device__ static __forceinline__ int addr(int line, int pos) { return line * PITCH + (pos ^ ((pos >> 4) & 7)); }
};

// In-place stage (block length LB, radix R, sub-stride S = LB/R) of one item of one line.
// FWD (DIF): butterfly then twiddle w_LB^(k t);  inverse (DIT): conj twiddle then butterfly.
template <int N, int LB, int R, bool FWD, class Lay>
__device__ __forceinline__ void pstage_item_tw(float4 *sm, const float2 (&tw)[R], int line, int b) {
    constexpr int S = LB / R;
    const int t = b % S;
    const int base = (b / S) * LB + t;
    P2 v[R];
    if (FWD) {
#pragma unroll
        for (int j = 0; j < R; ++j) v[j] = lds_p2(sm + Lay::addr(line, base + j * S));
        pbfly<R, -1>(v);
#pragma unroll
        for (int i = 0; i < R; ++i) {
            const int k = brev(i, R);
            if (S > 1 && k > 0) v[i] = pmul(v[i], tw[k]);
        }
#pragma unroll
        for (int i = 0; i < R; ++i) sts_p2(sm + Lay::addr(line, base + brev(i, R) * S), v[i]);
    } else {
#pragma unroll
        for (int k = 0; k < R; ++k) v[k] = lds_p2(sm + Lay::addr(line, base + k * S));
        if (S > 1) pbfly_dit<R>(v, tw);
        else pbfly<R, +1>(v);
#pragma unroll
        for (int i = 0; i < R; ++i) sts_p2(sm + Lay::addr(line, base + brev(i, R) * S), v[i]);
    }
}
template <int N, int LB, int R, bool FWD, class Lay, bool TSM = false>
__device__ __forceinline__ void pstage_item(float4 *sm, const float2 *__restrict__ lut, int line, int b) {
    constexpr int S = LB / R;
    float2 tw[R];
    if (S > 1) load_tw<R, S, 1, TSM>(tw, lut, b % S);
    pstage_item_tw<N, LB, R, FWD, Lay>(sm, tw, line, b);
}
template <int N, int LB, int R, bool FWD, class Lay, int TPL, bool TSM = false>
__device__ __forceinline__ void pstage_line(float4 *sm, const float2 *__restrict__ lut, int line, int lt) {
    constexpr int NBL = N / R;
#pragma unroll 1
    for (int b = lt; b < NBL; b += TPL) pstage_item<N, LB, R, FWD, Lay, TSM>(sm, lut, line, b);
}

// Interleaved first/last-stage table: lutAB[k][t] = (A.x, B.x, A.y, B.y) with A = w_N^(k t) (even
// half) and B = w_2N^((2k+1) t) (odd half, carries the zero-padding twist; fft_engine.cuh).
template <int R, int S>
__device__ __forceinline__ void load_tw_ab(float2 (&wre)[R], float2 (&wim)[R], const float4 *__restrict__ lut, int t) {
#pragma unroll
    for (int k = 0; k < R; ++k) {
        const float4 f = __ldg(lut + k * S + t);
        wre[k] = make_float2(f.x, f.y);
        wim[k] = make_float2(f.z, f.w);
    }
}

// First forward stage from registers: x[j] is the input at position t + j*S1 (natural order).
// even half: FFT of x; odd half: FFT of x w_2N^pos (the constant part w_(2 R1)^j applied here).
template <int N, int R1, class Lay>
__device__ __forceinline__ void pfirst_fwd_tw(const float2 (&x)[R1], int line, int t, float4 *sm,
                                              const float2 (&wre)[R1], const float2 (&wim)[R1]) {
    constexpr int S1 = N / R1;
    P2 v[R1];
#pragma unroll
    for (int j = 0; j < R1; ++j) {
        const float2 o = j > 0 ? mul_w32<-1>(x[j], j * (16 / R1)) : x[j];
        v[j] = P2{make_float2(x[j].x, o.x), make_float2(x[j].y, o.y)};
    }
    pbfly<R1, -1>(v);
#pragma unroll
    for (int i = 0; i < R1; ++i) v[i] = pmul2(v[i], wre[brev(i, R1)], wim[brev(i, R1)]);
#pragma unroll
    for (int i = 0; i < R1; ++i) sts_p2(sm + Lay::addr(line, t + brev(i, R1) * S1), v[i]);
}

// Periodic (unpadded) form: the two lanes of a value are two independent lines A and B (adjacent rows in k_row,
// adjacent columns in k_conv) that share every twiddle; xa, xb are their inputs at position t + j*S1.  The
// table passed as wre/wim holds w_N^(k t) in both lanes.
template <int N, int R1, class Lay>
__device__ __forceinline__ void pfirst_fwd_2l(const float2 (&xa)[R1], const float2 (&xb)[R1], int line, int t, float4 *sm,
                                              const float2 (&wre)[R1], const float2 (&wim)[R1]) {
    constexpr int S1 = N / R1;
    P2 v[R1];
#pragma unroll
    for (int j = 0; j < R1; ++j) v[j] = P2{make_float2(xa[j].x, xb[j].x), make_float2(xa[j].y, xb[j].y)};
    pbfly<R1, -1>(v);
#pragma unroll
    for (int i = 0; i < R1; ++i) v[i] = pmul2(v[i], wre[brev(i, R1)], wim[brev(i, R1)]);
#pragma unroll
    for (int i = 0; i < R1; ++i) sts_p2(sm + Lay::addr(line, t + brev(i, R1) * S1), v[i]);
}
// Last inverse stage of the periodic form: za[j], zb[j] = IFFT_N of line A, B at position t + j*S1.
template <int N, int R1, class Lay>
__device__ __forceinline__ void plast_inv_2l(float2 (&za)[R1], float2 (&zb)[R1], int line, int t, const float4 *sm,
                                             const float2 (&wre)[R1], const float2 (&wim)[R1]) {
    constexpr int S1 = N / R1;
    P2 v[R1];
#pragma unroll
    for (int k = 0; k < R1; ++k) v[k] = lds_p2(sm + Lay::addr(line, t + k * S1));
    pbfly_dit<R1>(v, wre, wim);
#pragma unroll
    for (int i = 0; i < R1; ++i) {
        const int j = brev(i, R1);
        za[j] = make_float2(v[i].re.x, v[i].im.x);
        zb[j] = make_float2(v[i].re.y, v[i].im.y);
    }
}

template <int N, int R1, class Lay>
__device__ __forceinline__ void pfirst_fwd(const float2 (&x)[R1], int line, int t, float4 *sm,
                                           const float4 *__restrict__ lutAB) {
    float2 wre[R1], wim[R1];
    load_tw_ab<R1, N / R1>(wre, wim, lutAB, t);
    pfirst_fwd_tw<N, R1, Lay>(x, line, t, sm, wre, wim);
}

// Last inverse stage into registers, both halves combined (inverse of pfirst_fwd followed by the
// crop): z[j] = IFFT_N(even half)[pos] + conj(w_2N^pos) IFFT_N(odd half)[pos], pos = t + j*S1.
template <int N, int R1, class Lay>
__device__ __forceinline__ void plast_inv_tw(float2 (&z)[R1], int line, int t, const float4 *sm,
                                             const float2 (&wre)[R1], const float2 (&wim)[R1]) {
    constexpr int S1 = N / R1;
    P2 v[R1];
#pragma unroll
    for (int k = 0; k < R1; ++k) v[k] = lds_p2(sm + Lay::addr(line, t + k * S1));
    pbfly_dit<R1>(v, wre, wim);
#pragma unroll
    for (int i = 0; i < R1; ++i) {
        const int j = brev(i, R1);
        const float2 o = mul_w32<+1>(make_float2(v[i].re.y, v[i].im.y), j * (16 / R1));
        z[j] = make_float2(v[i].re.x + o.x, v[i].im.x + o.y);
    }
}

template <int N, int R1, class Lay>
__device__ __forceinline__ void plast_inv(float2 (&z)[R1], int line, int t, const float4 *sm,
                                          const float4 *__restrict__ lutAB) {
    float2 wre[R1], wim[R1];
    load_tw_ab<R1, N / R1>(wre, wim, lutAB, t);
    plast_inv_tw<N, R1, Lay>(z, line, t, sm, wre, wim);
}

// Fused middle of the convolution: last forward stage (contiguous blocks of RL), multiply by ghat,
// first inverse stage, in registers (north_star: "pointwise G multiply fused into the last forward
// and first inverse butterfly stage").  With e = eps/k0^2 and alpha = (|p|^2/k0^2 - 1)/e,
//   k0^2 ghat = 1/(e (alpha - i)) = (alpha + i) / (e (alpha^2 + 1))
// so v ghat = ((v.re alpha - v.im) + i (v.im alpha + v.re)) / (alpha^2 + 1): six packed operations
// and one MUFU.RCP per half; the constant 1/(e k0^2) rides on the normalisation applied by k_row.
// p2x2: the line-axis table |p|^2/(e k0^2), interleaved over the halves, [j][block] float2 = (even, odd);
// a_line: (|p|^2 of the other axes / k0^2 - 1) / e, per lane (equal lanes for a padded line; the two columns'
// values in the periodic form).
template <int N, int RL, bool TSM>
__device__ __forceinline__ void load_p2x2(float2 (&pp)[RL], const float2 *__restrict__ p2x2, int b) {
#pragma unroll
    for (int j = 0; j < RL; ++j) pp[j] = TSM ? p2x2[j * (N / RL) + b] : __ldg(p2x2 + j * (N / RL) + b);
}
// Parameters of the k-space multiplier potential of Eq. 24, non-dimensional:
//   VV(k)/k0^2 = -i A kappa^nu + B kappa^(nu+1) - i e,  kappa = k/k0,  A = tau w k0^(nu-2),  B = eta k0^(nu-1).
struct KAbs {
    float A, B, nu, e;
};

// KABS = true: the spectrum of the (unmultiplied) term is multiplied by ghat(p) VV(|p|) instead of ghat(p)
// (homogeneous absorbing-dispersive medium, Eq. 24); kappa^2 = 1 + e alpha comes from the same tables.
// TWOF = true: lane 0 holds F[U_s u], lane 1 F[u]: lane 0 <- ghat (lane 0 + VV lane 1), lane 1 <- 0.
template <int N, int RL, class Lay, bool TSM = false, bool KABS = false, bool TWOF = false>
__device__ __forceinline__ void pmid_conv_item(float4 *sm, int line, int b, const float2 *__restrict__ p2x2,
                                               float2 a_line, KAbs ka = KAbs{0.f, 0.f, 0.f, 0.f}) {
    const int base = b * RL;
    float2 pp[RL];
    load_p2x2<N, RL, TSM>(pp, p2x2, b);
    P2 v[RL];
#pragma unroll
    for (int j = 0; j < RL; ++j) v[j] = lds_p2(sm + Lay::addr(line, base + j));
    pbfly<RL, -1>(v);
    P2 u[RL];
    if (!KABS) {
        // u[k] = X[k] (alpha + i) r, r = 1/(alpha^2 + 1), goes straight into the inverse butterfly: the r of a
        // second operand is folded into the first layer (s = a + t r, d = a - t r), so t r is never formed.
        constexpr int h = RL / 2;
        float2 rr[h];
#pragma unroll
        for (int i = 0; i < RL; ++i) {
            const int k = brev(i, RL);
            const float2 al = __fadd2_rn(pp[k], a_line);
            const float2 d = __ffma2_rn(al, al, f2(1.0f));
            const float2 r = make_float2(rcp_fast(d.x), rcp_fast(d.y));
            const P2 t = P2{__ffma2_rn(v[i].re, al, neg2(v[i].im)), __ffma2_rn(v[i].im, al, v[i].re)};
            if (k < h) {
                u[k] = P2{__fmul2_rn(t.re, r), __fmul2_rn(t.im, r)};
            } else {
                u[k] = t;
                rr[k - h] = r;
            }
        }
        int pend[RL];
#pragma unroll
        for (int m = 0; m < h; ++m) {
            const P2 a = u[m], t = u[m + h];
            u[m] = P2{__ffma2_rn(t.re, rr[m], a.re), __ffma2_rn(t.im, rr[m], a.im)};
            u[m + h] = P2{__ffma2_rn(t.re, neg2(rr[m]), a.re), __ffma2_rn(t.im, neg2(rr[m]), a.im)};
            pend[m] = 0;
            pend[m + h] = m * (8 / h);
        }
        pbfly_layers<RL, +1, RL / 4>(u, pend);
    } else {
#pragma unroll
        for (int i = 0; i < RL; ++i) {
            const int k = brev(i, RL);
            const float2 al = __fadd2_rn(pp[k], a_line);
            const float2 d = __ffma2_rn(al, al, f2(1.0f));
            const float2 r = make_float2(rcp_fast(d.x), rcp_fast(d.y));
            P2 w = P2{__fmul2_rn(__ffma2_rn(v[i].re, al, neg2(v[i].im)), r), __fmul2_rn(__ffma2_rn(v[i].im, al, v[i].re), r)};
            if (KABS && ka.nu > 0.f) {
                // kappa^nu = exp2(nu/2 log2(kappa^2)); frequencies masked for the periodic boundary (alpha ~ 1e18) give 0
                float2 q = __ffma2_rn(al, f2(ka.e), f2(1.0f));  // kappa^2 = |p|^2/k0^2 (>= 0 up to rounding)
                q = make_float2(fmaxf(q.x, 0.f), fmaxf(q.y, 0.f));
                const float2 lg = make_float2(__log2f(q.x), __log2f(q.y));
                const float2 kn = make_float2(exp2f(0.5f * ka.nu * lg.x), exp2f(0.5f * ka.nu * lg.y));
                const float2 k1 = make_float2(exp2f(0.5f * lg.x), exp2f(0.5f * lg.y));
                const float2 ok = make_float2(al.x < 1.0e17f ? 1.f : 0.f, al.y < 1.0e17f ? 1.f : 0.f);
                float2 vr = __fmul2_rn(__fmul2_rn(__fmul2_rn(kn, k1), f2(ka.B)), ok);                    // Re VV/k0^2
                float2 vi = __fmul2_rn(neg2(__ffma2_rn(kn, f2(ka.A), f2(ka.e))), ok);                    // Im VV/k0^2
                if (TWOF) { vr.x = 1.f; vi.x = 0.f; }   // lane 0 carries the spatial term: no multiplier
                w = P2{__ffma2_rn(w.re, vr, neg2(__fmul2_rn(w.im, vi))), __ffma2_rn(w.re, vi, __fmul2_rn(w.im, vr))};
            }
            if (TWOF) w = P2{make_float2(w.re.x + w.re.y, 0.f), make_float2(w.im.x + w.im.y, 0.f)};
            u[k] = w;
        }
        pbfly<RL, +1>(u);
    }
#pragma unroll
    for (int i = 0; i < RL; ++i) sts_p2(sm + Lay::addr(line, base + brev(i, RL)), u[i]);
}

}  // namespace tbs
