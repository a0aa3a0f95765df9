// dispatch.cuh -- launch configurations per transform length and run-time dispatch.
#pragma once
#include "kernels.cuh"

namespace tbs {

// Column-tile kernels: T adjacent lines per CTA, NT threads.  Shared memory = 2*N*T*8 bytes
// (both parity halves of the padded line).
template <int N> struct ColCfg;
template <> struct ColCfg<32>   { static constexpr int T = 16, NT = 64;  };
template <> struct ColCfg<64>   { static constexpr int T = 16, NT = 128; };
template <> struct ColCfg<128>  { static constexpr int T = 16, NT = 128; };
template <> struct ColCfg<256>  { static constexpr int T = 16, NT = 256; };
template <> struct ColCfg<512>  { static constexpr int T = 8,  NT = 512; };
template <> struct ColCfg<1024> { static constexpr int T = 8,  NT = 512; };
#ifndef TBS_COL2048_T
#define TBS_COL2048_T 4
#define TBS_COL2048_NT 512
#endif
template <int T_, int NT_> struct ColCfgT { static constexpr int T = T_, NT = NT_; };
template <> struct ColCfg<2048> : ColCfgT<TBS_COL2048_T, TBS_COL2048_NT> {};
template <> struct ColCfg<4096> { static constexpr int T = 2,  NT = 512; };

// Row kernels: ROWS rows per CTA, NT threads, at least MINB CTAs per SM (register cap).  Shared memory = 2*ROWS*(N + N/16)*8 bytes.
template <int N> struct RowCfg;
template <> struct RowCfg<32> { static constexpr int ROWS = 16, NT = 64, MINB = 4; };
template <> struct RowCfg<64> { static constexpr int ROWS = 8, NT = 64, MINB = 4; };
template <> struct RowCfg<128> { static constexpr int ROWS = 8, NT = 64, MINB = 4; };
template <> struct RowCfg<256> { static constexpr int ROWS = 4, NT = 64, MINB = 4; };
template <> struct RowCfg<512> { static constexpr int ROWS = 2, NT = 128, MINB = 4; };
template <> struct RowCfg<1024> { static constexpr int ROWS = 2, NT = 128, MINB = 3; };
#ifndef TBS_ROW2048_ROWS
#define TBS_ROW2048_ROWS 2
#define TBS_ROW2048_NT 256
#define TBS_ROW2048_MINB 2
#endif
template <int R_, int NT_, int MB_> struct RowCfgT { static constexpr int ROWS = R_, NT = NT_, MINB = MB_; };
template <> struct RowCfg<2048> : RowCfgT<TBS_ROW2048_ROWS, TBS_ROW2048_NT, TBS_ROW2048_MINB> {};
template <> struct RowCfg<4096> { static constexpr int ROWS = 1, NT = 256, MINB = 2; };

template <int N, int MODE>
static cudaError_t launch_col_t(const ColArgs &a, int n_outer, cudaStream_t st, bool set_attr) {
    using C = ColCfg<N>;
    constexpr size_t smem = 2 * (size_t)N * C::T * sizeof(float2);
    auto kern = k_col<N, C::T, C::NT, MODE>;
    if (set_attr) return cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    const unsigned grid = (unsigned)(n_outer * (a.inner_len / C::T));
    kern<<<grid, C::NT, smem, st>>>(a);
    return cudaGetLastError();
}

template <int MODE>
static cudaError_t launch_col(int N, const ColArgs &a, int n_outer, cudaStream_t st, bool set_attr = false) {
    switch (N) {
        case 32:   return launch_col_t<32, MODE>(a, n_outer, st, set_attr);
        case 64:   return launch_col_t<64, MODE>(a, n_outer, st, set_attr);
        case 128:  return launch_col_t<128, MODE>(a, n_outer, st, set_attr);
        case 256:  return launch_col_t<256, MODE>(a, n_outer, st, set_attr);
        case 512:  return launch_col_t<512, MODE>(a, n_outer, st, set_attr);
        case 1024: if (MODE == MODE_CONV) return launch_col_t<1024, MODE_CONV>(a, n_outer, st, set_attr); break;
        case 2048: if (MODE == MODE_CONV) return launch_col_t<2048, MODE_CONV>(a, n_outer, st, set_attr); break;
        case 4096: if (MODE == MODE_CONV) return launch_col_t<4096, MODE_CONV>(a, n_outer, st, set_attr); break;
        default: break;
    }
    return cudaErrorInvalidValue;
}

template <int N, bool FIRST>
static cudaError_t launch_row_t(const RowArgs &a, cudaStream_t st, bool set_attr) {
    using C = RowCfg<N>;
    constexpr size_t smem = 2 * (size_t)C::ROWS * RowLay<N>::PITCH * sizeof(float2);
    auto kern = k_row<N, C::ROWS, C::NT, C::MINB, FIRST>;
    if (set_attr) return cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    kern<<<(unsigned)(a.rows / C::ROWS), C::NT, smem, st>>>(a);
    return cudaGetLastError();
}

template <bool FIRST>
static cudaError_t launch_row(int N, const RowArgs &a, cudaStream_t st, bool set_attr = false) {
    switch (N) {
        case 32:   return launch_row_t<32, FIRST>(a, st, set_attr);
        case 64:   return launch_row_t<64, FIRST>(a, st, set_attr);
        case 128:  return launch_row_t<128, FIRST>(a, st, set_attr);
        case 256:  return launch_row_t<256, FIRST>(a, st, set_attr);
        case 512:  return launch_row_t<512, FIRST>(a, st, set_attr);
        case 1024: return launch_row_t<1024, FIRST>(a, st, set_attr);
        case 2048: return launch_row_t<2048, FIRST>(a, st, set_attr);
        case 4096: return launch_row_t<4096, FIRST>(a, st, set_attr);
        default: break;
    }
    return cudaErrorInvalidValue;
}

static inline void radices_of(int N, int &r1, int &r2, int &rl) {
    switch (N) {
        case 32:   r1 = Radix<32>::R1;   r2 = Radix<32>::R2;   rl = Radix<32>::RL;   break;
        case 64:   r1 = Radix<64>::R1;   r2 = Radix<64>::R2;   rl = Radix<64>::RL;   break;
        case 128:  r1 = Radix<128>::R1;  r2 = Radix<128>::R2;  rl = Radix<128>::RL;  break;
        case 256:  r1 = Radix<256>::R1;  r2 = Radix<256>::R2;  rl = Radix<256>::RL;  break;
        case 512:  r1 = Radix<512>::R1;  r2 = Radix<512>::R2;  rl = Radix<512>::RL;  break;
        case 1024: r1 = Radix<1024>::R1; r2 = Radix<1024>::R2; rl = Radix<1024>::RL; break;
        case 2048: r1 = Radix<2048>::R1; r2 = Radix<2048>::R2; rl = Radix<2048>::RL; break;
        default:   r1 = Radix<4096>::R1; r2 = Radix<4096>::R2; rl = Radix<4096>::RL; break;
    }
}

}  // namespace tbs
