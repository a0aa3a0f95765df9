// fft_engine.cuh -- in-place shared-memory FFT building blocks for the TBS kernels (sm_100a).
//
// A length-N complex FFT (N = 2^n, 32..4096) is factored as N = R1 * [R2] * RL with radices in
// {4, 8, 16}.  Forward transforms are decimation-in-frequency (natural order in, digit-reversed
// order out), inverse transforms are the mirrored decimation-in-time (digit-reversed in, natural
// out), so no reorder pass ever runs: the Green's spectrum ghat(p) is even in every
// component of p and is simply indexed in the scrambled order (tables are built in "position
// order" on the host).  Data lives in shared memory between stages; every stage reads and writes
// the same positions ("in place"), so one barrier of the threads that own the line separates two
// stages.  This file holds the scalar form (k_col) and what both forms share; fft_engine_x2.cuh holds
// the packed form (k_row, k_conv).
//
// Zero padding N -> M = 2N (BASELINE.json north_star) is never materialised:
//   X[2k+s] = sum_{j<N} (x[j] w_M^{js}) w_N^{jk}            (forward, s = 0, 1: two length-N FFTs)
//   y[j]    = sum_s w_M^{-js} IFFT_N(Y[2k+s])[j],  j < N     (inverse followed by the crop)
// so a padded line is stored as two halves of N "positions": P = s*N + pos.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

namespace tbs {

// ---- complex helpers -------------------------------------------------------------------------
__device__ __forceinline__ float2 cadd(float2 a, float2 b) { return make_float2(a.x + b.x, a.y + b.y); }
__device__ __forceinline__ float2 csub(float2 a, float2 b) { return make_float2(a.x - b.x, a.y - b.y); }
__device__ __forceinline__ float2 cmul(float2 a, float2 b) {
    return make_float2(a.x * b.x - a.y * b.y, a.x * b.y + a.y * b.x);
}
// a * conj(b)
__device__ __forceinline__ float2 cmulc(float2 a, float2 b) {
    return make_float2(a.x * b.x + a.y * b.y, a.y * b.x - a.x * b.y);
}

// ---- asynchronous copies (global -> shared) -------------------------------------------------------
// Row tiles are contiguous in global memory and come in with one bulk copy (TMA engine, completion
// on an mbarrier); column tiles are N short segments and come in with 16-byte cp.async (LDGSTS).
__device__ __forceinline__ uint32_t smem_u32(const void *p) { return (uint32_t)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void mbar_init(uint64_t *b, int count) {
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(b)), "r"(count) : "memory");
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
}
__device__ __forceinline__ void mbar_expect_tx(uint64_t *b, uint32_t bytes) {
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(b)), "r"(bytes) : "memory");
}
__device__ __forceinline__ void bulk_g2s(void *dst, const void *src, uint32_t bytes, uint64_t *b) {
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];"
                 ::"r"(smem_u32(dst)), "l"(src), "r"(bytes), "r"(smem_u32(b)) : "memory");
}
// 2-D tiled TMA load (cp.async.bulk.tensor): box at element coordinates (c0, c1) of the tensor map.
__device__ __forceinline__ void tma_load_2d(void *dst, const void *tmap, int c0, int c1, uint64_t *b) {
    asm volatile("cp.async.bulk.tensor.2d.shared::cluster.global.tile.mbarrier::complete_tx::bytes [%0], [%1, {%2, %3}], [%4];"
                 ::"r"(smem_u32(dst)), "l"(tmap), "r"(c0), "r"(c1), "r"(smem_u32(b)) : "memory");
}
// 2-D tiled TMA store of a dense shared-memory box; completion tracked by the bulk async-group.
__device__ __forceinline__ void tma_store_2d(const void *tmap, const void *src, int c0, int c1) {
    asm volatile("cp.async.bulk.tensor.2d.global.shared::cta.tile.bulk_group [%0, {%1, %2}], [%3];"
                 ::"l"(tmap), "r"(c0), "r"(c1), "r"(smem_u32(src)) : "memory");
}
__device__ __forceinline__ void bulk_commit() { asm volatile("cp.async.bulk.commit_group;" ::: "memory"); }
__device__ __forceinline__ void bulk_wait_read() { asm volatile("cp.async.bulk.wait_group.read 0;" ::: "memory"); }
__device__ __forceinline__ void bulk_wait_all() { asm volatile("cp.async.bulk.wait_group 0;" ::: "memory"); }
__device__ __forceinline__ void fence_async_smem() { asm volatile("fence.proxy.async.shared::cta;" ::: "memory"); }
__device__ __forceinline__ void mbar_wait(uint64_t *b, uint32_t parity) {
    uint32_t ok;
    do {
        asm volatile("{ .reg .pred p; mbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2; selp.u32 %0, 1, 0, p; }"
                     : "=r"(ok) : "r"(smem_u32(b)), "r"(parity) : "memory");
    } while (!ok);
}
__device__ __forceinline__ void cp_async16(void *dst, const void *src) {
    asm volatile("cp.async.cg.shared.global [%0], [%1], 16;" ::"r"(smem_u32(dst)), "l"(src) : "memory");
}
__device__ __forceinline__ void cp_async_commit() { asm volatile("cp.async.commit_group;" ::: "memory"); }
__device__ __forceinline__ void cp_async_wait_all() { asm volatile("cp.async.wait_group 0;" ::: "memory"); }
// Programmatic dependent launch: let the next kernel of the stream be scheduled while this one drains / wait
// for the previous kernel of the stream to complete and its writes to be visible (no-ops without the attribute).
__device__ __forceinline__ void griddep_launch() { asm volatile("griddepcontrol.launch_dependents;" ::: "memory"); }
__device__ __forceinline__ void griddep_wait() { asm volatile("griddepcontrol.wait;" ::: "memory"); }
// Streaming accesses of the fields (read or written once per term): keep them out of L1, which holds the tables.
__device__ __forceinline__ float2 ld_stream(const float2 *p) {
    float2 v;
    asm volatile("ld.global.L1::no_allocate.v2.f32 {%0, %1}, [%2];" : "=f"(v.x), "=f"(v.y) : "l"(p));
    return v;
}
__device__ __forceinline__ float2 ld_stream_nc(const float2 *p) {
    float2 v;
    asm volatile("ld.global.nc.L1::no_allocate.v2.f32 {%0, %1}, [%2];" : "=f"(v.x), "=f"(v.y) : "l"(p));
    return v;
}
__device__ __forceinline__ void prefetch_l2(const void *p) { asm volatile("prefetch.global.L2 [%0];" ::"l"(p)); }

// ---- radix plan ------------------------------------------------------------------------------
template <int N> struct Radix;
template <> struct Radix<32>   { static constexpr int R1 = 8,  R2 = 0,  RL = 4;  };
template <> struct Radix<64>   { static constexpr int R1 = 8,  R2 = 0,  RL = 8;  };
template <> struct Radix<128>  { static constexpr int R1 = 16, R2 = 0,  RL = 8;  };
template <> struct Radix<256>  { static constexpr int R1 = 16, R2 = 0,  RL = 16; };
template <> struct Radix<512>  { static constexpr int R1 = 8,  R2 = 8,  RL = 8;  };
template <> struct Radix<1024> { static constexpr int R1 = 8,  R2 = 8,  RL = 16; };
template <> struct Radix<2048> { static constexpr int R1 = 8,  R2 = 16, RL = 16; };
template <> struct Radix<4096> { static constexpr int R1 = 16, R2 = 16, RL = 16; };

// bit reversal of i within log2(R) bits
__host__ __device__ constexpr int brev(int i, int R) {
    int r = 0;
    for (int b = 1; b < R; b <<= 1) { r = (r << 1) | (i & 1); i >>= 1; }
    return r;
}

// ---- radix-R butterfly in registers ----------------------------------------------------------
// d * w_16^(idx16) with sign SGN (SGN = -1: exp(-2 pi i idx/16), forward; +1: inverse).
template <int SGN>
__device__ __forceinline__ float2 mul_w16(float2 d, int idx16) {
    constexpr float C1 = 0.92387953251128674f;  // cos(pi/8)
    constexpr float S1 = 0.38268343236508977f;  // sin(pi/8)
    constexpr float H = 0.70710678118654752f;   // sqrt(1/2)
    const float s = (float)SGN;
    switch (idx16) {
        case 0: return d;
        case 1: return make_float2(d.x * C1 - s * d.y * S1, d.y * C1 + s * d.x * S1);
        case 2: return make_float2((d.x - s * d.y) * H, (d.y + s * d.x) * H);
        case 3: return make_float2(d.x * S1 - s * d.y * C1, d.y * S1 + s * d.x * C1);
        case 4: return make_float2(-s * d.y, s * d.x);
        case 5: return make_float2(-d.x * S1 - s * d.y * C1, -d.y * S1 + s * d.x * C1);
        case 6: return make_float2((-d.x - s * d.y) * H, (-d.y + s * d.x) * H);
        default: return make_float2(-d.x * C1 - s * d.y * S1, -d.y * C1 + s * d.x * S1);
    }
}

// DFT_R of v (sign SGN), natural order in, BIT-REVERSED order out: v[i] <- X[brev(i, R)].
template <int R, int SGN>
__device__ __forceinline__ void bfly(float2 (&v)[R]) {
#pragma unroll
    for (int h = R / 2; h >= 1; h >>= 1) {
#pragma unroll
        for (int g = 0; g < R; g += 2 * h) {
#pragma unroll
            for (int m = 0; m < h; ++m) {
                float2 a = v[g + m], b = v[g + m + h];
                v[g + m] = cadd(a, b);
                v[g + m + h] = mul_w16<SGN>(csub(a, b), m * (8 / h));
            }
        }
    }
}

// ---- per-stage twiddle look-up tables ---------------------------------------------------------
// A stage with block length LB = R*S needs w_LB^(k t), k < R, for its sub-index t < S.  The tables
// are stored k-major, [R][S] (float2), so that the threads of a warp -- consecutive t -- fetch each
// twiddle with one contiguous 256-byte load (built in double by k_stage_lut, setup_kernels.cuh):
//   lutA[k][t] = w_N^(k t)            first / last stage, even-frequency half (parity 0)
//   lutB[k][t] = w_2N^((2k+1) t)      first / last stage, odd-frequency half  (parity 1): the
//                                     zero-padding twist w_2N^(pos), pos = t + j*S1, factors into
//                                     w_2N^t (folded into the table) and the constant w_(2 R1)^j
//   lutC[k][t] = w_S1^(k t)           middle stage (three-stage plans only)
struct Luts {
    const float2 *A, *B, *C;
    const float4 *AB;  // A and B interleaved (fft_engine_x2.cuh)
};

// K0 = 1 skips k = 0 (the twiddle is 1 in tables A and C).
// SM = true: the table is a shared-memory copy (plain loads); false: global memory through L1.
template <int R, int S, int K0, bool SM = false>
__device__ __forceinline__ void load_tw(float2 (&w)[R], const float2 *__restrict__ lut, int t) {
#pragma unroll
    for (int k = K0; k < R; ++k) w[k] = SM ? lut[k * S + t] : __ldg(lut + k * S + t);
}

// d * w_32^(idx) with sign SGN; idx in [0, 16).
template <int SGN>
__device__ __forceinline__ float2 mul_w32(float2 d, int idx) {
    constexpr float C[16] = {1.0f, 0.98078528040323043f, 0.92387953251128674f, 0.83146961230254524f,
                             0.70710678118654752f, 0.55557023301960218f, 0.38268343236508977f,
                             0.19509032201612825f, 0.0f, -0.19509032201612825f, -0.38268343236508977f,
                             -0.55557023301960218f, -0.70710678118654752f, -0.83146961230254524f,
                             -0.92387953251128674f, -0.98078528040323043f};
    constexpr float S[16] = {0.0f, 0.19509032201612825f, 0.38268343236508977f, 0.55557023301960218f,
                             0.70710678118654752f, 0.83146961230254524f, 0.92387953251128674f,
                             0.98078528040323043f, 1.0f, 0.98078528040323043f, 0.92387953251128674f,
                             0.83146961230254524f, 0.70710678118654752f, 0.55557023301960218f,
                             0.38268343236508977f, 0.19509032201612825f};
    if (idx == 0) return d;
    if (idx == 8) return make_float2(-(float)SGN * d.y, (float)SGN * d.x);
    const float c = C[idx], s = (float)SGN * S[idx];
    return make_float2(d.x * c - d.y * s, d.y * c + d.x * s);
}
// x[j] *= w_(2R)^(SGN j): the constant part of the zero-padding twist of the odd-frequency half.
template <int R, int SGN>
__device__ __forceinline__ void twist_const(float2 (&x)[R]) {
#pragma unroll
    for (int j = 1; j < R; ++j) x[j] = mul_w32<SGN>(x[j], j * (16 / R));
}

// ---- shared-memory layouts -------------------------------------------------------------------
// Column tile: T adjacent lines interleaved, [pos][T].  A warp covers 32/T positions x T lines.
// XOR swizzle of the low position bits keeps the contiguous-block stage (stride RL between
// lanes) conflict-free for T < 16.
template <int N, int T_, int RL>
struct ColLay {
    static constexpr int T = T_;
    static constexpr int G = (16 / T_ > 1) ? 16 / T_ : 1;
    static constexpr int SMEM_ELEMS = N * T_;
    __device__ static __forceinline__ int addr(int line, int pos) {
        if (G > 1) pos ^= (pos / RL) & (G - 1);
        return pos * T_ + line;
    }
    template <int NBL>
    __device__ static __forceinline__ void split(int w, int &line, int &b) { line = w % T_; b = w / T_; }
};
// Threads that own one line in the line-group kernels (k_row, k_conv): one radix-16 item each in
// the widest stage.  Groups of TPL >= 32 threads synchronise on a named barrier of their own,
// smaller groups share a warp and use __syncwarp, so no stage waits for the whole CTA.
// Byte offset of k_conv's staging buffer behind its work area, rounded to the 1024-byte swizzle atom.
__host__ __device__ constexpr int conv_stage_offset(int N, int T) {
    return (T * N * 16 + 1023) / 1024 * 1024;
}
// k_conv shared memory: work area, staging, the middle-stage twiddle table C (N/R1 entries, plans with
// three stages) and -- when that leaves the CTA under 128 KB, so that L1 keeps room for the first/last-
// stage table (measured: at N = 2048 the copy costs more in L1 misses than it saves) -- the line-axis table.
__host__ __device__ constexpr int conv_lutc_entries(int N) { return N >= 512 ? N / 8 : 0; }
__host__ __device__ constexpr bool conv_p2_in_smem(int N, int T) {
    return conv_stage_offset(N, T) + N * T * 8 + conv_lutc_entries(N) * 8 + N * 8 <= 128 * 1024;
}
__host__ __device__ constexpr int conv_smem_bytes(int N, int T) {
    return conv_stage_offset(N, T) + N * T * 8 + conv_lutc_entries(N) * 8 + (conv_p2_in_smem(N, T) ? N * 8 : 0);
}
// the periodic form of k_conv (T/2 line slots per tile, no table copies)
__host__ __device__ constexpr int conv_smem_bytes_per(int N, int T) { return conv_stage_offset(N, T / 2) + N * T * 8; }
__host__ __device__ constexpr int tpl_of(int N) { return N / 16 >= 4 ? N / 16 : 4; }
// k_conv: first/last-stage items per line >= threads of two lines (N = 512, 1024, 2048): the fused last/first
// stage runs by line pairs with 16-byte accesses to the tile buffer.
__host__ __device__ constexpr bool conv_pair_exchange(int N) { return N == 512 || N == 1024 || N == 2048; }
// k_row: threads per row, and whether the W row is staged by a bulk copy a tile ahead.  N = 4096 runs two
// items per thread and reads W directly: with the 64 KB staging buffer only one row would fit an SM.
__host__ __device__ constexpr int row_tpl_of(int N) { return N == 4096 ? 128 : tpl_of(N); }
__host__ __device__ constexpr bool row_staged(int N) { return N < 4096; }
// Middle stage (radix R2, blocks of R2*RL, stride RL) and contiguous stage (blocks of RL) touch the same RL x RL
// block from the same 16 threads when R2 == RL and both deal item b to thread b mod TPL: a warp barrier is
// enough between them (the plans of N = 2048 and 4096).
__host__ __device__ constexpr bool warp_local_mid(int R2, int RL, int TPL) {
    return R2 > 0 && R2 == RL && RL == 16 && TPL >= 32 && TPL % 32 == 0;
}
template <int GT>
__device__ __forceinline__ void group_sync(int gid) {
    if (GT <= 32) __syncwarp();
    else asm volatile("bar.sync %0, %1;" ::"r"(gid + 1), "n"(GT) : "memory");
}

// ---- in-place stages on shared memory, both parity halves at once --------------------------------
// sm holds the even-frequency half at [0, HALF) and the odd-frequency half at [HALF, 2 HALF); one
// work item is the pair of butterflies (parity 0, parity 1) at the same (line, block, t), which
// share their twiddles.  Block length LB, radix R, sub-stride S = LB/R.
// FWD (DIF): butterfly then twiddle w_LB^(k t);  inverse (DIT): conj twiddle then butterfly.
template <int N, int LB, int R, bool FWD, class Lay, int HALF>
__device__ __forceinline__ void stage_item(float2 *sm, const float2 *__restrict__ lut, int line, int b) {
    constexpr int S = LB / R;
    const int t = b % S;
    const int base = (b / S) * LB + t;
    float2 tw[R];
    if (S > 1) load_tw<R, S, 1>(tw, lut, t);
#pragma unroll
    for (int p = 0; p < 2; ++p) {
        float2 *s = sm + p * HALF;
        float2 v[R];
        if (FWD) {
#pragma unroll
            for (int j = 0; j < R; ++j) v[j] = s[Lay::addr(line, base + j * S)];
            bfly<R, -1>(v);
#pragma unroll
            for (int i = 0; i < R; ++i) {
                const int k = brev(i, R);
                float2 o = v[i];
                if (S > 1 && k > 0) o = cmul(o, tw[k]);
                s[Lay::addr(line, base + k * S)] = o;
            }
        } else {
#pragma unroll
            for (int k = 0; k < R; ++k) {
                float2 x = s[Lay::addr(line, base + k * S)];
                if (S > 1 && k > 0) x = cmulc(x, tw[k]);
                v[k] = x;
            }
            bfly<R, +1>(v);
#pragma unroll
            for (int i = 0; i < R; ++i) s[Lay::addr(line, base + brev(i, R) * S)] = v[i];
        }
    }
}
// all lines of a CTA tile, items dealt round-robin to the NT threads
template <int N, int LB, int R, bool FWD, class Lay, int NT, int HALF>
__device__ __forceinline__ void stage_pair(float2 *sm, const float2 *__restrict__ lut, int tid, int total) {
    constexpr int NBL = N / R;
    for (int w = tid; w < total; w += NT) {
        int line, b;
        Lay::template split<NBL>(w, line, b);
        stage_item<N, LB, R, FWD, Lay, HALF>(sm, lut, line, b);
    }
}
// First forward stage from registers: x[j] is the input at position t + j*S1 (natural order).
// Writes the even-frequency half (FFT of x) and the odd-frequency half (FFT of x w_2N^pos).
template <int N, int R1, class Lay, int HALF>
__device__ __forceinline__ void first_fwd_pair(const float2 (&x)[R1], int line, int t, float2 *sm,
                                               const Luts &L) {
    constexpr int S1 = N / R1;
    float2 tw[R1];
    float2 v[R1];
    load_tw<R1, S1, 1>(tw, L.A, t);
#pragma unroll
    for (int j = 0; j < R1; ++j) v[j] = x[j];
    bfly<R1, -1>(v);
#pragma unroll
    for (int i = 0; i < R1; ++i) {
        const int k = brev(i, R1);
        sm[Lay::addr(line, t + k * S1)] = k > 0 ? cmul(v[i], tw[k]) : v[i];
    }
    load_tw<R1, S1, 0>(tw, L.B, t);
#pragma unroll
    for (int j = 0; j < R1; ++j) v[j] = x[j];
    twist_const<R1, -1>(v);
    bfly<R1, -1>(v);
#pragma unroll
    for (int i = 0; i < R1; ++i) {
        const int k = brev(i, R1);
        sm[HALF + Lay::addr(line, t + k * S1)] = cmul(v[i], tw[k]);
    }
}

// Last inverse stage into registers, both halves combined (inverse of first_fwd_pair followed by
// the crop): z[j] = IFFT_N(even half)[pos] + conj(w_2N^pos) IFFT_N(odd half)[pos], pos = t + j*S1.
template <int N, int R1, class Lay, int HALF>
__device__ __forceinline__ void last_inv_pair(float2 (&z)[R1], int line, int t, const float2 *sm,
                                              const Luts &L) {
    constexpr int S1 = N / R1;
    float2 tw[R1];
    float2 v[R1], u[R1];
    load_tw<R1, S1, 1>(tw, L.A, t);
#pragma unroll
    for (int k = 0; k < R1; ++k) {
        const float2 a = sm[Lay::addr(line, t + k * S1)];
        v[k] = k > 0 ? cmulc(a, tw[k]) : a;
    }
    bfly<R1, +1>(v);
    load_tw<R1, S1, 0>(tw, L.B, t);
#pragma unroll
    for (int k = 0; k < R1; ++k) u[k] = cmulc(sm[HALF + Lay::addr(line, t + k * S1)], tw[k]);
    bfly<R1, +1>(u);
#pragma unroll
    for (int i = 0; i < R1; ++i) {
        const int j = brev(i, R1);
        z[j] = cadd(v[i], mul_w32<+1>(u[i], j * (16 / R1)));
    }
}

// 1/d by MUFU.RCP (rcp.approx: relative error <= 2^-23), without the IEEE-division slow path.
__device__ __forceinline__ float rcp_fast(float d) {
    float r;
    asm("rcp.approx.ftz.f32 %0, %1;" : "=f"(r) : "f"(d));
    return r;
}

}  // namespace tbs
