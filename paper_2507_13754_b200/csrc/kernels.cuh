// kernels.cuh -- the Born-term kernels, built on fft_engine.cuh.
//
//   k_row  (K1 / K3+K1 fused, "K31"): per grid row along x.
//          inverse half:  W row (2N positions) -> IFFT_x -> crop -> u = A.(.) -> p (+)= u,
//                         partial ||u||^2, ||p||^2 -> last CTA finalises r_n and the stop flag
//          forward half:  w = V.u (or the source S for term 0) -> zero-pad -> FFT_x -> W row
//          u never leaves the chip between the two halves (cross-term fusion).
//   k_conv: per tile of T adjacent lines along a strided axis (y in 2-D, z in 3-D): pad, FFT, .ghat,
//          IFFT, crop, in place (K2 in 2-D, the z pass in 3-D); tiles move by TMA.
//   k_col<MODE> (3-D y passes, scalar engine):
//          FWD : pad, FFT  N -> 2N positions
//          INV : IFFT, crop  2N positions -> N
// Both parity halves of a padded line (fft_engine.cuh) are resident in shared memory at once, so
// the input is read once and the twiddles of a butterfly pair are fetched once.  k_row and k_conv
// use the packed engine of fft_engine_x2.cuh (both halves in one register pair).
#pragma once
#include <cuda.h>  // CUtensorMap (type only; the encoder is fetched through the runtime, tbs.cu)

#include "fft_engine_x2.cuh"

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
    unsigned int next_tile;  // k_row: row tiles handed out beyond the first one of every group
    // divergence guard (the paper only caps the iterations, and states that
    // convergence needs ||GV|| < 1)
    int hold;        // 1: never stop (tbs_profile_term times kernels on a series that may overflow)
    int rising;      // consecutive terms with r_n above 10 x its running minimum
    double rmin;     // running minimum of r_n, n >= 1
    double uu0;      // ||u_0||^2
};
// r_n above 10 x its minimum for this many consecutive terms, or ||u_n|| above GROWTH_LIMIT ||u_0||: diverged
constexpr int DIVERGE_RISING_TERMS = 32;
constexpr double DIVERGE_GROWTH_SQ = 1.0e12;  // (1e6)^2 on the squared norms

enum { MODE_FWD = 1, MODE_INV = 2 };

struct ColArgs {
    const float2 *in;
    float2 *out;
    long long in_line_stride, out_line_stride;    // between consecutive positions of a line
    long long in_outer_stride, out_outer_stride;  // between consecutive outer indices
    int inner_len;                                // number of adjacent lines (multiple of T)
    int n_outer;                                  // number of outer indices
    const float2 *p2_line;  // [N] (even, odd) |p|^2/eps of the line axis, order of pmid_conv_item
    const float *p2_inner;  // [inner_len] of the inner (x) axis, position order  (CONV)
    const float *p2_outer;  // [n_outer] of the outer axis or nullptr             (CONV)
    float inv_e;            // k0^2/eps = 1/damping
    KAbs kabs;              // k-space multiplier potential of Eq. 24 (k_conv<..., KABS = true> only)
    int masked;             // periodic boundary: axis tables mask the odd padded frequencies (general k_conv)
    int per;                // 1: periodic boundary, unpadded form (k_conv<..., PER>; 2-D); 2: its two-field form (TWOF)
    Luts lut;
    const Ctl *ctl;
};

// Persistent: each CTA walks tiles blockIdx.x, blockIdx.x + gridDim.x, ...  For FWD the N input
// positions of the next tile are fetched with cp.async into a staging buffer while the current
// tile computes.
template <int N, int T, int NT, int MODE>
__global__ void __launch_bounds__(NT) k_col(ColArgs a) {
    using P = Radix<N>;
    constexpr int R1 = P::R1, R2 = P::R2, RL = P::RL;
    constexpr int R2s = R2 > 0 ? R2 : 2;
    constexpr int S1 = N / R1;
    static_assert((S1 * T) % NT == 0 && NT % T == 0, "tile/thread mismatch");
    static_assert(T % 2 == 0, "16-byte staging copies need an even tile width");
    constexpr int NB = (S1 * T) / NT;  // first/last-stage butterfly pairs per thread
    constexpr int TSTEP = NT / T;
    constexpr int HALF = N * T;
    using Lay = ColLay<N, T, RL>;
    extern __shared__ __align__(1024) float2 sm[];
    float2 *stg = sm + 2 * HALF;  // [N][T] staged input tile (FWD)
    griddep_launch();
    griddep_wait();
    if (a.ctl->done) return;

    const int tid = threadIdx.x;
    const int line = tid % T, t0 = tid / T;
    const int tiles = a.inner_len / T;
    const int total = tiles * a.n_outer;

    auto stage_tile = [&](int tile) {
        const int inner0 = (tile % tiles) * T;
        const int outer = tile / tiles;
        const float2 *src = a.in + (long long)outer * a.in_outer_stride + inner0;
        constexpr int CPR = T / 2;  // 16-byte chunks per position
        for (int c = tid; c < N * CPR; c += NT) {
            const int r = c / CPR, cc = c % CPR;
            cp_async16(stg + r * T + 2 * cc, src + (long long)r * a.in_line_stride + 2 * cc);
        }
        cp_async_commit();
    };
    if (MODE != MODE_INV && (int)blockIdx.x < total) stage_tile(blockIdx.x);

    for (int tile = blockIdx.x; tile < total; tile += gridDim.x) {
        const int inner0 = (tile % tiles) * T;
        const int outer = tile / tiles;
        const float2 *in = a.in + (long long)outer * a.in_outer_stride + inner0 + line;
        float2 *out = a.out + (long long)outer * a.out_outer_stride + inner0 + line;

        // ---- forward: N inputs -> both halves in smem ----
        if (MODE != MODE_INV) {
            cp_async_wait_all();
            __syncthreads();  // staged tile visible; previous tile's readers of the work area are done
#pragma unroll
            for (int i = 0; i < NB; ++i) {
                const int t = t0 + i * TSTEP;
                float2 x[R1];
#pragma unroll
                for (int j = 0; j < R1; ++j) x[j] = stg[(t + j * S1) * T + line];
                first_fwd_pair<N, R1, Lay, HALF>(x, line, t, sm, a.lut);
            }
            __syncthreads();
            if (tile + (int)gridDim.x < total) stage_tile(tile + gridDim.x);
            if (R2 > 0) {
                stage_pair<N, S1, R2s, true, Lay, NT, HALF>(sm, a.lut.C, tid, (N / R2s) * T);
                __syncthreads();
            }
        }
        if (MODE == MODE_FWD) {
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
            continue;
        } else {
            // INV: first inverse stage straight from global
            __syncthreads();  // previous tile's readers of the work area are done
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
    float scale;          // k0^2/(eps prod(2 n)): inverse-transform normalisation and the 1/e of ghat (k_conv)
    int crit_row;         // >= 0: convergence measure of PAPER.md:258-260 Eq. 30 on this row (L1, previous field);
                          // < 0: full-grid L2, ||u_n|| / ||p_n|| (reading A8)
    float2 *ucbs;         // CBS scheme: [rows][N] current term u_n (read and replaced); nullptr for TBS
    float inv_e;          // CBS: k0^2/eps
    int do_fwd;           // 0: stop after the inverse half (tbs_apply_green)
    int per;              // 1: periodic boundary, unpadded form (k_row<..., PER>): W is [rows][N]; 2: two-field form (TWOF)
    double *norms;        // [max_terms+1][2] sum |u|^2, sum |p|^2
    double *history;      // [max_terms+1]
    Ctl *ctl;
    Luts lut;
};

// ---------------------------------------------------------------------------------------------------
// Line-group kernels.  A line (a grid row for k_row, a column for k_conv) is owned by TPL = N/16
// threads for the whole of its transform; those threads synchronise among themselves only (named
// barrier, or __syncwarp when several lines share a warp), so the shared-memory traffic of one
// group overlaps the butterflies of another instead of every stage waiting for the whole CTA.
// ---------------------------------------------------------------------------------------------------

// Layout of a W row along x (2N complex values): the parity halves are interleaved and the last
// digit is transposed, so that every access of k_row is a 16-byte-per-lane, lane-contiguous one:
//   column c = 2 q + s,  q = k * (N/RL) + b   <->   half s, position pos = b * RL + k
// (b = block of the contiguous last forward / first inverse stage, k = index inside the block).
// The x axis table of the Green's spectrum is built in this column order (k_axis_table).
//
// FIRST = true : forward half only, w = src * src_scale (term 0: u_0 = G S, Eq. 20)
// FIRST = false: inverse half (K3) + forward half (K1) of the next term
// GEN   = true : the general variant: the convergent Born series update (a.ucbs) and/or
//                the one-row L1 criterion of Eq. 30 (a.crit_row >= 0), chosen at run time; GEN = false is
//                the hot path (traditional series, full-grid L2 measure) without either
// Persistent and group-independent: group G of CTA B walks row tiles (B*GROUPS + G) + i*gridDim.x*
// GROUPS; the W rows of its next tile arrive by one bulk copy (completion on the group's mbarrier)
// in a staging buffer while the current tile computes.
// PER = true: the periodic (unpadded) form (Eq. 19, Alg. 1 l.36-38): one length-N transform per grid
// row, W is [rows][N], and the two lanes of every packed value are two adjacent grid rows (a line slot = rows
// 2s, 2s + 1); first/last-stage table with w_N^(k t) in both lanes, no padding twist, no crop.
// TWOF = true (periodic boundary with the k-space multiplier potential AND a spatial scatterer term): the two lanes
// are two FIELDS of the same grid row, U_s u_n and u_n, transformed together so that k_conv can form
// ghat (F[U_s u_n] + VV F[u_n]) (Eq. 24 plus the U_s term of Eq. 25); W keeps the padded layout (column 2q + h =
// field h at x-frequency q); only lane 0 comes back from the inverse transform.
template <int N, int GROUPS, int MINB, bool FIRST, bool GEN, bool PER = false, bool TWOF = false>
__global__ void __launch_bounds__(GROUPS * (row_tpl_of(N) >= 32 ? row_tpl_of(N) : 32), MINB) k_row(RowArgs a) {
    static_assert(!(PER && TWOF), "one meaning of the lanes at a time");
    using P = Radix<N>;
    constexpr int R1 = P::R1, R2 = P::R2, RL = P::RL;
    constexpr int R2s = R2 > 0 ? R2 : 2;
    constexpr int S1 = N / R1;
    constexpr int NBL = N / RL;
    constexpr int M = 2 * N;
    constexpr int TPL = row_tpl_of(N);
    constexpr bool STAGED = row_staged(N);
    constexpr int GR = TPL >= 32 ? 1 : 32 / TPL;  // rows per group
    constexpr int GT = TPL * GR;                   // threads per group
    constexpr int NT = GROUPS * GT;
    constexpr int ROWS = GROUPS * GR;
    constexpr int NITEM = S1 / TPL;  // first/last-stage items per thread
    static_assert(S1 % TPL == 0, "items per thread");
    constexpr bool EARLY = !PER && NITEM * R1 <= 16;  // p and V requested a barrier ahead (else per item: registers)
    constexpr int NR = PER ? 2 : 1;  // grid rows per line slot
    // R2 == RL: the RL x RL block a middle-stage item works in is the block of the RL contiguous-stage items of the
    // same 16 threads (item b of either stage lies in block b / RL), so the two stages only need a warp barrier.
    constexpr bool WL = warp_local_mid(R2, RL, TPL);
    using Lay = LineLay<N>;
    extern __shared__ __align__(1024) float2 sm[];
    float4 *wk = reinterpret_cast<float4 *>(sm);  // [ROWS][PITCH] work area, both halves per slot
    float4 *stg = wk + ROWS * Lay::PITCH;         // [ROWS][N] staged W rows
    __shared__ float red[2][32];
    __shared__ __align__(8) uint64_t mbar[GROUPS];
    __shared__ int next_gt[GROUPS];
    griddep_launch();
    griddep_wait();
    if (a.ctl->done) return;

    const int tid = threadIdx.x;
    const int g = tid / GT, gl = tid % GT;
    const int l = g * GR + gl / TPL;  // CTA-local line
    const int lt = gl % TPL;
    const int ngt = a.rows / (GR * NR);  // group tiles
    const int gstride = gridDim.x * GROUPS;
    const int term = FIRST ? 0 : a.ctl->term;
    constexpr uint32_t TILE_BYTES = (uint32_t)GR * M * sizeof(float2);
    uint32_t phase = 0;
    float uu = 0.f, pp = 0.f;

    int gt = blockIdx.x * GROUPS + g;
    if (!FIRST) {
        if (tid == 0)
            for (int i = 0; i < GROUPS; ++i) mbar_init(&mbar[i], 1);
        __syncthreads();
        if (STAGED && gl == 0 && gt < ngt) {
            mbar_expect_tx(&mbar[g], TILE_BYTES);
            bulk_g2s(stg + g * GR * N, a.W + (long long)gt * GR * M, TILE_BYTES, &mbar[g]);
        }
    }

    // Every group starts on tile B*GROUPS + G; further tiles are handed out by an atomic counter (the
    // groups of a launch do not finish their rows at the same pace; FIRST keeps the static walk).
#pragma unroll 1
    while (gt < ngt) {
        const int row = gt * GR + gl / TPL;   // line slot: grid row `row` (padded form), rows 2 row, 2 row + 1 (periodic)
        float wrow[NR];
        float2 pold[EARLY ? NITEM : 1][R1], vpot[EARLY ? NITEM : 1][R1];
#pragma unroll
        for (int h = 0; h < NR; ++h) wrow[h] = a.scale;
        if (!FIRST) {
            // ---------------- inverse half: IFFT_x, crop, window, accumulate ----------------
            // pull the p and V rows of this tile towards L2 while the W rows arrive
            for (int i = gl; i < GR * NR * N / 16; i += GT) {
                prefetch_l2(a.p + (long long)gt * GR * NR * N + i * 16);
                prefetch_l2(a.V + (long long)gt * GR * NR * N + i * 16);
                if (GEN && a.ucbs) prefetch_l2(a.ucbs + (long long)gt * GR * NR * N + i * 16);
            }
#pragma unroll
            for (int h = 0; h < NR; ++h) {
                wrow[h] *= __ldg(&a.ay[(row * NR + h) % a.ny]);
                if (a.az) wrow[h] *= __ldg(&a.az[(row * NR + h) / a.ny]);
            }
            if (STAGED) {
                mbar_wait(&mbar[g], phase);
                phase ^= 1u;
            }
            const float4 *wrow_g = reinterpret_cast<const float4 *>(a.W + (long long)row * M);
            // first inverse stage (contiguous blocks of RL) from the staged rows
#pragma unroll 1
            for (int b = lt; b < NBL; b += TPL) {
                P2 v[RL];
#pragma unroll
                for (int k = 0; k < RL; ++k) {
                    if (PER) {
                        // rows A and B of the slot lie one behind the other (N values each)
                        const float2 *ra = STAGED ? reinterpret_cast<const float2 *>(stg + l * N)
                                                  : reinterpret_cast<const float2 *>(wrow_g);
                        const float2 fa = ra[k * NBL + b], fb = ra[N + k * NBL + b];
                        v[k] = P2{make_float2(fa.x, fb.x), make_float2(fa.y, fb.y)};
                    } else {
                        const float4 f = STAGED ? stg[l * N + k * NBL + b] : wrow_g[k * NBL + b];
                        v[k] = P2{make_float2(f.x, f.z), make_float2(f.y, f.w)};
                    }
                }
                pbfly<RL, +1>(v);
#pragma unroll
                for (int i = 0; i < RL; ++i) sts_p2(wk + Lay::addr(l, b * RL + brev(i, RL)), v[i]);
            }
            // the group's staging rows are free once every thread of the group is past this point: take the next
            // tile and fetch its W rows
            auto fetch_next = [&]() {
                if (gl == 0) {
                    const int nxt = gstride + (int)atomicAdd(&a.ctl->next_tile, 1u);
                    next_gt[g] = nxt;
                    if (STAGED && nxt < ngt) {
                        mbar_expect_tx(&mbar[g], TILE_BYTES);
                        bulk_g2s(stg + g * GR * N, a.W + (long long)nxt * GR * M, TILE_BYTES, &mbar[g]);
                    }
                }
            };
            if (WL) {
                __syncwarp();
            } else {
                group_sync<GT>(g);
                fetch_next();
            }
            if (R2 > 0) pstage_line<N, S1, R2s, false, Lay, TPL>(wk, a.lut.C, l, lt);
            // request the running field and the potential at the thread's output points now: their
            // latency passes under the barrier and the shared-memory loads of the last inverse stage
            if (EARLY) {
#pragma unroll
                for (int it = 0; it < NITEM; ++it)
#pragma unroll
                    for (int j = 0; j < R1; ++j) {
                        const long long gi = (long long)row * N + lt + it * TPL + j * S1;
                        pold[it][j] = term > 0 ? ld_stream(&a.p[gi]) : make_float2(0.f, 0.f);
                        vpot[it][j] = ld_stream_nc(&a.V[gi]);
                    }
            }
            if (R2 > 0) group_sync<GT>(g);
            if (WL) fetch_next();
        }
        // last inverse stage + crop + window + accumulate + V.u + first forward stage; a thread
        // writes the slots it has just read, so the items need no barrier between them.  The p and V
        // values of all items of the thread were requested before the barrier in front of this stage.
#pragma unroll
        for (int it = 0; it < NITEM; ++it) {
            const int t = lt + it * TPL;
            // x[h][j]: line h of the slot (the one padded line, or the two grid rows of the periodic form) at
            // position t + j*S1 -- first the inverse transform's output, then the input of the forward half
            float2 x[NR][R1];
            float2 xf[R1];  // TWOF: lane 1 -- the inverse transform's unused lane, then the field u itself
            float2 wre[R1], wim[R1];
            load_tw_ab<R1, S1>(wre, wim, a.lut.AB, t);
            constexpr int pi = EARLY ? 1 : 0;
            const int ii = it * pi;  // slot of this item's p and V values
            if (!FIRST) {
                if (PER) plast_inv_2l<N, R1, Lay>(x[0], x[NR - 1], l, t, wk, wre, wim);
                else if (TWOF) plast_inv_2l<N, R1, Lay>(x[0], xf, l, t, wk, wre, wim);
                else plast_inv_tw<N, R1, Lay>(x[0], l, t, wk, wre, wim);
            }
#pragma unroll
            for (int h = 0; h < NR; ++h) {
                const int grow = row * NR + h;  // grid row
                if (FIRST) {
#pragma unroll
                    for (int j = 0; j < R1; ++j) {
                        const float2 v = ld_stream_nc(&a.src[(long long)grow * N + t + j * S1]);
                        x[h][j] = make_float2(v.x * a.src_scale, v.y * a.src_scale);
                        if (TWOF) xf[j] = make_float2(0.f, 0.f);  // term 0 is u_0 = A G S: nothing for the multiplier
                    }
                    continue;
                }
                if (!EARLY) {
#pragma unroll
                    for (int j = 0; j < R1; ++j) {
                        const long long gi = (long long)grow * N + t + j * S1;
                        pold[0][j] = term > 0 ? ld_stream(&a.p[gi]) : make_float2(0.f, 0.f);
                        vpot[0][j] = ld_stream_nc(&a.V[gi]);
                    }
                }
                // The run-time options of the general variant are tested around whole loops over the R1
                // outputs, never inside them: the loop bodies stay branch-free and interleave.
                float2 uv[R1];
#pragma unroll
                for (int j = 0; j < R1; ++j) {
                    const float wgt = wrow[h] * __ldg(&a.ax[t + j * S1]);
                    uv[j] = make_float2(x[h][j].x * wgt, x[h][j].y * wgt);
                }
                if (GEN && a.ucbs) {
                    // convergent Born series: u_{n+1} = u_n + gamma (A G(V u_n) - u_n), gamma = i V / eps
#pragma unroll
                    for (int j = 0; j < R1; ++j) {
                        const long long gi = (long long)grow * N + t + j * S1;
                        const float2 gam = make_float2(-vpot[ii][j].y * a.inv_e, vpot[ii][j].x * a.inv_e);
                        const float2 uo = term > 0 ? a.ucbs[gi] : make_float2(0.f, 0.f);
                        uv[j] = cadd(uo, cmul(gam, csub(uv[j], uo)));
                        a.ucbs[gi] = uv[j];
                    }
                }
                if (!GEN || a.crit_row < 0) {
#pragma unroll
                    for (int j = 0; j < R1; ++j) {
                        const float2 pv = cadd(pold[ii][j], uv[j]);
                        a.p[(long long)grow * N + t + j * S1] = pv;
                        uu = fmaf(uv[j].x, uv[j].x, fmaf(uv[j].y, uv[j].y, uu));
                        pp = fmaf(pv.x, pv.x, fmaf(pv.y, pv.y, pp));
                    }
                } else if (grow != a.crit_row) {
#pragma unroll
                    for (int j = 0; j < R1; ++j) a.p[(long long)grow * N + t + j * S1] = cadd(pold[ii][j], uv[j]);
                } else {
                    // Eq. 30: sum |psi_{l+1} - psi_l| and sum |psi_l| on one row; moduli through a 2^20 pre-scale
                    // (the squares stay in range for 1e-25 < |.| < 1e13)
                    constexpr float SC = 1048576.f, ISC = 1.f / 1048576.f;
#pragma unroll
                    for (int j = 0; j < R1; ++j) {
                        const float2 po = pold[ii][j];
                        a.p[(long long)grow * N + t + j * S1] = cadd(po, uv[j]);
                        const float ax = uv[j].x * SC, ay = uv[j].y * SC, bx = po.x * SC, by = po.y * SC;
                        uu = fmaf(sqrtf(fmaf(ax, ax, ay * ay)), ISC, uu);
                        pp = fmaf(sqrtf(fmaf(bx, bx, by * by)), ISC, pp);
                    }
                }
#pragma unroll
                for (int j = 0; j < R1; ++j) {
                    x[h][j] = cmul(vpot[ii][j], uv[j]);
                    if (TWOF) xf[j] = uv[j];
                }
            }
            if (!FIRST && !a.do_fwd) continue;
            if (PER) pfirst_fwd_2l<N, R1, Lay>(x[0], x[NR - 1], l, t, wk, wre, wim);
            else if (TWOF) pfirst_fwd_2l<N, R1, Lay>(x[0], xf, l, t, wk, wre, wim);
            else pfirst_fwd_tw<N, R1, Lay>(x[0], l, t, wk, wre, wim);
        }
        group_sync<GT>(g);
        const int gt_next = FIRST ? gt + gstride : next_gt[g];
        if (!FIRST && !a.do_fwd) {
            gt = gt_next;
            continue;
        }
        // ---------------- forward half: the remaining stages of FFT_x ----------------
        if (R2 > 0) {
            pstage_line<N, S1, R2s, true, Lay, TPL>(wk, a.lut.C, l, lt);
            if (WL) __syncwarp();
            else group_sync<GT>(g);
        }
        // last forward stage (contiguous blocks of RL) straight to global memory.  A thread reads
        // exactly the slots it writes in the first inverse stage of its next tile.
#pragma unroll 1
        for (int b = lt; b < NBL; b += TPL) {
            P2 v[RL];
#pragma unroll
            for (int j = 0; j < RL; ++j) v[j] = lds_p2(wk + Lay::addr(l, b * RL + j));
            pbfly<RL, -1>(v);
            if (PER) {
                float2 *ga = a.W + (long long)row * M + b;
#pragma unroll
                for (int i = 0; i < RL; ++i) {
                    ga[brev(i, RL) * NBL] = make_float2(v[i].re.x, v[i].im.x);
                    ga[N + brev(i, RL) * NBL] = make_float2(v[i].re.y, v[i].im.y);
                }
            } else {
                float4 *gp = reinterpret_cast<float4 *>(a.W + (long long)row * M) + b;
#pragma unroll
                for (int i = 0; i < RL; ++i)
                    gp[brev(i, RL) * NBL] = make_float4(v[i].re.x, v[i].im.x, v[i].re.y, v[i].im.y);
            }
        }
        if (FIRST) group_sync<GT>(g);  // the next tile's first stage writes slots other threads still read
        gt = gt_next;
    }

    if (!FIRST) {
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
                const double r = (!GEN || a.crit_row < 0) ? sqrt(nu) / sqrt(np) : (term == 0 ? 1.0 : nu / np);
                a.history[term] = (term == 0) ? 1.0 : r;
                a.ctl->ticket = 0;
                a.ctl->next_tile = 0;
                a.ctl->n_terms = term;
                a.ctl->term = term + 1;
                // divergence guard: a non-finite measure; the term norm a million times that of u_0 (L2 measure);
                // the measure above ten times its minimum for 32 terms in a row
                bool diverged = !(r == r) || r > 1.0e300;
                if (term == 0) {
                    a.ctl->uu0 = nu;
                    a.ctl->rmin = 1.0e300;
                    a.ctl->rising = 0;
                } else if (!diverged) {
                    if ((!GEN || a.crit_row < 0) && nu > DIVERGE_GROWTH_SQ * a.ctl->uu0) diverged = true;
                    const double rmin = a.ctl->rmin;
                    if (r < rmin) a.ctl->rmin = r;
                    const int rising = r > 10.0 * rmin ? a.ctl->rising + 1 : 0;
                    a.ctl->rising = rising;
                    if (rising >= DIVERGE_RISING_TERMS) diverged = true;
                }
                if (a.ctl->hold) {
                    // profiling: keep going whatever the values
                } else if (diverged) {
                    a.ctl->done = 1; a.ctl->status = -5;
                } else if (term >= 1 && r < a.ctl->tol) {
                    a.ctl->done = 1; a.ctl->status = 0;
                } else if (term >= a.ctl->max_terms) {
                    a.ctl->done = 1; a.ctl->status = 1;
                }
            }
        }
    }
}

// K2 (2-D) / the z pass (3-D): for each of T adjacent lines along a strided axis: pad, FFT, .ghat,
// IFFT, crop, in place in global memory.  Persistent.  Tiles move by TMA through one
// tile buffer used in place for both directions; the last inverse stage of a tile is fused with the
// first forward stage of the next one (as in k_row), so a tile costs four stages and ONE CTA-wide
// barrier; between them the T line groups run on their own barriers.
//
// PER = true: the periodic (unpadded) form of the paper itself (Eq. 19, Alg. 1 l.36-38): one
// length-N transform per column, and the two lanes of every packed value are the two columns of a 16-byte chunk
// of the tile -- T/2 line slots per tile, the tile buffer read and written 16 bytes at a time, half the columns
// and half the arithmetic per column of the padded form.  2-D only (a.p2_outer is not read).
// TWOF = true (with PER): the two columns of a chunk are the two fields of k_row<..., TWOF> at one x-frequency; the
// fused stage multiplies lane 1 by VV as well, adds it to lane 0 and clears it.
template <int N, int T, int MINB, bool KABS, bool PER = false, bool TWOF = false>
__global__ void __launch_bounds__((PER ? T / 2 : T) * tpl_of(N), MINB) k_conv(ColArgs a, const __grid_constant__ CUtensorMap tmap) {
    static_assert(!TWOF || (PER && KABS), "the two-field form runs on the periodic kernels with the multiplier");
    using P = Radix<N>;
    constexpr int R1 = P::R1, R2 = P::R2, RL = P::RL;
    constexpr int R2s = R2 > 0 ? R2 : 2;
    constexpr int S1 = N / R1;
    constexpr int TPL = tpl_of(N);
    constexpr int NL = PER ? T / 2 : T;  // line slots of a tile
    constexpr int NT = NL * TPL;
    constexpr int GT = TPL >= 32 ? TPL : 32;
    static_assert(T % 2 == 0 && NT % 32 == 0, "tile shape");
    constexpr int CPR = T / 2;  // 16-byte chunks (line pairs) per position
    constexpr bool WL = warp_local_mid(R2, RL, TPL);  // see k_row
    // fused last/first stage by line pairs (see there): when the stage has an item for every thread of two lines
    constexpr bool PAIRX = !PER && conv_pair_exchange(N) && (2 * TPL) % 32 == 0 && T / 2 <= 7;
    using Lay = LineLay<N>;
    extern __shared__ __align__(1024) float2 sm[];
    float4 *wk = reinterpret_cast<float4 *>(sm);  // [T][PITCH] work area, both halves per slot
    // Staged input tile, position-major like global memory: [N][CPR] chunks of 16 bytes (lines 2c,
    // 2c+1), the chunk index XOR-swizzled with the position (the TMA swizzle mode of that row width)
    // so that the 8-byte reads of a line group (consecutive positions) are 2-way at worst.
    float4 *stg = wk + conv_stage_offset(N, NL) / 16;  // 1024-byte aligned (TMA swizzle atom)
    __shared__ __align__(8) uint64_t mbar;
    // Shared-memory copies of the tables every tile re-reads, for the tile shapes that leave room
    // (fft_engine.cuh, conv_p2_in_smem): the middle-stage twiddles C and the line-axis spectrum table.
    constexpr bool P2SM = !PER && conv_p2_in_smem(N, T);
    constexpr bool CSM = !PER && R2 > 0;  // the middle-stage table is small (N/R1 entries): always copied
    float2 *lutC_s = reinterpret_cast<float2 *>(stg + N * CPR);
    float2 *p2_s = lutC_s + conv_lutc_entries(N);
    griddep_launch();

    const int tid = threadIdx.x;
    // Two lines per warp (TPL = 16): quarter-warps alternate between the lines, so that the 8-byte accesses of a
    // half-warp to the tile buffer (lines 2c, 2c + 1 at 8 consecutive positions) fill whole 16-byte chunks --
    // conflict-free, where 16 positions of one line are 2-way.  The 16-byte work-area accesses go by quarter-warp
    // and see the same pattern either way.
    constexpr bool QW = TPL == 16 && !PER;
    const int line = QW ? (tid >> 5) * 2 + ((tid >> 3) & 1) : tid / TPL;
    const int lt = QW ? (tid & 7) + ((tid >> 4) & 1) * 8 : tid % TPL;
    const int g = tid / GT;
    const int tiles = a.inner_len / T;
    const int total = tiles * a.n_outer;
    auto swz = [](int r) { return CPR > 1 ? (r / (CPR >= 8 ? 1 : 8 / CPR)) % CPR : 0; };

    // A tile arrives as N/BR boxes of BR rows x T columns through the tensor map (cp.async.bulk.tensor,
    // hardware swizzle = the XOR above), issued by one thread, completion on mbar; the result leaves the
    // same way from the same buffer.
    constexpr int BR = N < 256 ? N : 256;
    constexpr uint32_t TILE_BYTES = (uint32_t)N * T * sizeof(float2);
    uint32_t phase = 0;
    auto tma_tile = [&](int tile) {
        mbar_expect_tx(&mbar, TILE_BYTES);
        const int c0 = (tile / tiles) * (int)a.in_outer_stride + (tile % tiles) * T;
#pragma unroll 1
        for (int k = 0; k < N / BR; ++k) tma_load_2d(stg + k * BR * CPR, &tmap, c0, k * BR, &mbar);
    };
    if (tid == 0) mbar_init(&mbar, 1);
    if (CSM)
        for (int i = tid; i < S1; i += NT) lutC_s[i] = __ldg(a.lut.C + i);
    if (P2SM)
        for (int i = tid; i < N; i += NT) p2_s[i] = __ldg(a.p2_line + i);
    const float2 *p2_tab = P2SM ? p2_s : a.p2_line;
    const float2 *lutC_tab = CSM ? lutC_s : a.lut.C;
    __syncthreads();
    // everything above reads plan constants only; the tiles and the stop flag are the previous kernel's
    griddep_wait();
    if (a.ctl->done) return;
    // I/O element of this thread's line at position r of the tile buffer
    float2 *io = reinterpret_cast<float2 *>(stg) + (line & 1);
    auto io_at = [&](int r) -> float2 & { return io[2 * (r * CPR + ((line >> 1) ^ swz(r)))]; };
    auto store_tile = [&](int tile) {
        const int c0 = (tile / tiles) * (int)a.out_outer_stride + (tile % tiles) * T;
#pragma unroll 1
        for (int k = 0; k < N / BR; ++k) tma_store_2d(&tmap, stg + k * BR * CPR, c0, k * BR);
        bulk_commit();
    };

    // The tile buffer serves both directions, in place: in the fused last/first stage a thread reads
    // the next tile's input at its positions and leaves the current tile's result there.  Thread 0
    // stores the buffer and refills it, once the store has been read out, for the tile after next:
    // under the first middle stage of the next tile (three-stage plans), else at once.
    int tile = blockIdx.x;
    if (tile >= total) return;
    if (tid == 0) tma_tile(tile);
    // ---- prologue: first stage of the first tile ----
    mbar_wait(&mbar, phase);
    phase ^= 1u;
#pragma unroll 1
    for (int t = lt; t < S1; t += TPL) {
        if (PER) {
            float2 wre[R1], wim[R1], xa[R1], xb[R1];
            load_tw_ab<R1, S1>(wre, wim, a.lut.AB, t);
#pragma unroll
            for (int j = 0; j < R1; ++j) {
                const int r = t + j * S1;
                const float4 f = stg[r * CPR + (line ^ swz(r))];
                xa[j] = make_float2(f.x, f.y);
                xb[j] = make_float2(f.z, f.w);
            }
            pfirst_fwd_2l<N, R1, Lay>(xa, xb, line, t, wk, wre, wim);
        } else {
            float2 x[R1];
#pragma unroll
            for (int j = 0; j < R1; ++j) x[j] = io_at(t + j * S1);
            pfirst_fwd<N, R1, Lay>(x, line, t, wk, a.lut.AB);
        }
    }
    __syncthreads();
    int to_load = tile + 2 * (int)gridDim.x < total ? tile + 2 * (int)gridDim.x : -1;  // refill after the next store
    if (tid == 0 && tile + (int)gridDim.x < total) tma_tile(tile + gridDim.x);

#pragma unroll 1
    for (; tile < total; tile += gridDim.x) {
        const int inner0 = (tile % tiles) * T;
        const int outer = tile / tiles;
        const bool more = tile + (int)gridDim.x < total;
        // alpha of a line from the other axes.  General variant (KABS): a line at a frequency the periodic
        // boundary masks (axis tables hold 1e18 there) gives exact zeros and is not computed.
        auto line_alpha_of = [&](int in0, int out, int ln) {
            float al = __ldg(&a.p2_inner[in0 + ln]) - 1.0f;
            if (a.p2_outer) al += __ldg(&a.p2_outer[out]);
            return al * a.inv_e;
        };
        auto line_alpha = [&](int in0, int out) { return line_alpha_of(in0, out, line); };
        float a_line = 0.f;
        if (KABS && !PER) a_line = line_alpha(inner0, outer);
        const bool dead = KABS && !PER && a_line > 1.0e17f;
        if (R2 > 0) {
            if (!dead) pstage_line<N, S1, R2s, true, Lay, TPL, CSM>(wk, lutC_tab, line, lt);
            if (WL) __syncwarp();
            else group_sync<GT>(g);  // by every line: lines of different state may share a warp
            // by now the store of the previous tile has been read out of the buffer: refill it
            if (tid == 0 && to_load >= 0 && tile != (int)blockIdx.x) {
                bulk_wait_read();
                tma_tile(to_load);
            }
            if (tile != (int)blockIdx.x) to_load = to_load >= 0 && to_load + (int)gridDim.x < total ? to_load + (int)gridDim.x : -1;
        }
        if (!dead) {
            if (!KABS) a_line = line_alpha(inner0, outer);
            float2 a_line2 = f2(a_line);
            // periodic form: the slot's two columns; the x table holds the N-grid value at entries 2q and 2q + 1
            if (PER) a_line2 = make_float2((__ldg(&a.p2_inner[(TWOF ? 1 : 2) * (inner0 + 2 * line)]) - 1.0f) * a.inv_e,
                                           (__ldg(&a.p2_inner[(TWOF ? 1 : 2) * (inner0 + 2 * line + 1)]) - 1.0f) * a.inv_e);
            KAbs ka = a.kabs;
            if (KABS && a.ctl->term == 0) ka.nu = 0.f;  // term 0 is u_0 = A G S: the plain Green's spectrum
#pragma unroll 1
            for (int b = lt; b < N / RL; b += TPL) pmid_conv_item<N, RL, Lay, P2SM, KABS, TWOF>(wk, line, b, p2_tab, a_line2, ka);
        }
        if (WL) __syncwarp();
        else group_sync<GT>(g);
        if (R2 > 0) {
            if (!dead) pstage_line<N, S1, R2s, false, Lay, TPL, CSM>(wk, lutC_tab, line, lt);
            if (!PAIRX) group_sync<GT>(g);
        }
        // pair exchange: the next stage reads both lines of the thread's pair
        if (PAIRX) asm volatile("bar.sync %0, %1;" ::"r"(8 + tid / (2 * TPL)), "n"(2 * TPL) : "memory");
        // ---- fused: last inverse stage of this tile, first forward stage of the next one ----
        if (more) {
            mbar_wait(&mbar, phase);
            phase ^= 1u;
        }
        bool dead_next = false;  // the same line of the next tile (another outer index in 3-D)
        if (KABS && !PER && more) {
            const int nt = tile + (int)gridDim.x;
            dead_next = line_alpha((nt % tiles) * T, nt / tiles) > 1.0e17f;
        }
        if (PER) {
#pragma unroll 1
            for (int t = lt; t < S1; t += TPL) {
                float2 wre[R1], wim[R1];
                load_tw_ab<R1, S1>(wre, wim, a.lut.AB, t);
                float2 za[R1], zb[R1], xa[R1], xb[R1];
                plast_inv_2l<N, R1, Lay>(za, zb, line, t, wk, wre, wim);
#pragma unroll
                for (int j = 0; j < R1; ++j) {
                    const int r = t + j * S1;
                    float4 &e = stg[r * CPR + (line ^ swz(r))];
                    const float4 f = e;
                    xa[j] = make_float2(f.x, f.y);
                    xb[j] = make_float2(f.z, f.w);
                    e = make_float4(za[j].x, za[j].y, zb[j].x, zb[j].y);
                }
                if (more) pfirst_fwd_2l<N, R1, Lay>(xa, xb, line, t, wk, wre, wim);
            }
        } else if (PAIRX) {
            // Pair exchange: a thread does this stage for BOTH lines of a 16-byte chunk of the tile buffer at its
            // positions, so the buffer is read and written 16 bytes at a time (conflict-free under the TMA swizzle,
            // half the instructions of the per-line 8-byte exchange) and the twiddles are fetched once per pair.
            const int l0 = 2 * (tid / (2 * TPL)), pt = tid % (2 * TPL);
            bool dp[2] = {false, false}, dn[2] = {false, false};
            if (KABS) {
                const int nt = tile + (int)gridDim.x;
#pragma unroll
                for (int q = 0; q < 2; ++q) {
                    dp[q] = line_alpha_of(inner0, outer, l0 + q) > 1.0e17f;
                    dn[q] = more && line_alpha_of((nt % tiles) * T, nt / tiles, l0 + q) > 1.0e17f;
                }
            }
#pragma unroll 1
            for (int t = pt; t < S1; t += 2 * TPL) {
                float2 wre[R1], wim[R1];
                load_tw_ab<R1, S1>(wre, wim, a.lut.AB, t);
                float4 xx[R1];
#pragma unroll
                for (int j = 0; j < R1; ++j) {
                    const int r = t + j * S1;
                    xx[j] = stg[r * CPR + ((l0 >> 1) ^ swz(r))];
                }
                float2 z0[R1], z1[R1], x[R1];
                if (!dp[0]) {
                    plast_inv_tw<N, R1, Lay>(z0, l0, t, wk, wre, wim);
                } else {
#pragma unroll
                    for (int j = 0; j < R1; ++j) z0[j] = make_float2(0.f, 0.f);
                }
                if (more && !dn[0]) {
#pragma unroll
                    for (int j = 0; j < R1; ++j) x[j] = make_float2(xx[j].x, xx[j].y);
                    pfirst_fwd_tw<N, R1, Lay>(x, l0, t, wk, wre, wim);
                }
                if (!dp[1]) {
                    plast_inv_tw<N, R1, Lay>(z1, l0 + 1, t, wk, wre, wim);
                } else {
#pragma unroll
                    for (int j = 0; j < R1; ++j) z1[j] = make_float2(0.f, 0.f);
                }
#pragma unroll
                for (int j = 0; j < R1; ++j) {
                    const int r = t + j * S1;
                    stg[r * CPR + ((l0 >> 1) ^ swz(r))] = make_float4(z0[j].x, z0[j].y, z1[j].x, z1[j].y);
                }
                if (more && !dn[1]) {
#pragma unroll
                    for (int j = 0; j < R1; ++j) x[j] = make_float2(xx[j].z, xx[j].w);
                    pfirst_fwd_tw<N, R1, Lay>(x, l0 + 1, t, wk, wre, wim);
                }
            }
        } else {
#pragma unroll 1
            for (int t = lt; t < S1; t += TPL) {
                float2 wre[R1], wim[R1];
                load_tw_ab<R1, S1>(wre, wim, a.lut.AB, t);
                float2 z[R1], x[R1];
                if (!dead) {
                    plast_inv_tw<N, R1, Lay>(z, line, t, wk, wre, wim);
                } else {
#pragma unroll
                    for (int j = 0; j < R1; ++j) z[j] = make_float2(0.f, 0.f);
                }
#pragma unroll
                for (int j = 0; j < R1; ++j) {
                    float2 &e = io_at(t + j * S1);
                    x[j] = e;
                    e = z[j];
                }
                if (more && !dead_next) pfirst_fwd_tw<N, R1, Lay>(x, line, t, wk, wre, wim);
            }
        }
        fence_async_smem();
        __syncthreads();  // result tile complete, next input consumed, next first stage in place
        if (tid == 0) {
            store_tile(tile);
            if (R2 == 0 && to_load >= 0) {  // two-stage plans: no stage to hide the drain under
                bulk_wait_read();
                tma_tile(to_load);
            }
        }
        if (R2 == 0) to_load = to_load >= 0 && to_load + (int)gridDim.x < total ? to_load + (int)gridDim.x : -1;
    }
    if (tid == 0) bulk_wait_all();
}

}  // namespace tbs
