// dispatch.cuh -- launch configurations per transform length and run-time dispatch.
#pragma once
#include "kernels.cuh"

namespace tbs {

// Column-tile kernel k_col (3-D y passes): T adjacent lines per CTA, NT threads.  Shared memory =
// 2*N*T*8 bytes (both parity halves of the padded line) + N*T*8 bytes of input staging (FWD).
template <int N> struct ColCfg;
template <> struct ColCfg<32>   { static constexpr int T = 16, NT = 64;  };
template <> struct ColCfg<64>   { static constexpr int T = 16, NT = 128; };
template <> struct ColCfg<128>  { static constexpr int T = 16, NT = 128; };
template <> struct ColCfg<256>  { static constexpr int T = 16, NT = 256; };
template <> struct ColCfg<512>  { static constexpr int T = 8,  NT = 512; };

// Row kernel k_row: GROUPS independent line groups per CTA (a group = N/16 threads on one row, or
// one warp on 32/(N/16) rows), at least MINB CTAs per SM (register cap).  Shared memory per row =
// N*16 bytes of work area + N*16 bytes of W staging (N = 4096: no staging, two items per thread).  Values measured on B200 (cfg2-cfg5).
template <int N> struct RowCfg { static constexpr int GROUPS = 4, MINB = 2; };   // N <= 512
template <> struct RowCfg<1024> { static constexpr int GROUPS = 2, MINB = 3; };
template <> struct RowCfg<2048> { static constexpr int GROUPS = 1, MINB = 3; };
template <> struct RowCfg<4096> { static constexpr int GROUPS = 1, MINB = 2; };

// Convolution kernel k_conv: T adjacent lines per CTA, T * max(N/16, 4) threads, at least MINB CTAs
// per SM.  Shared memory = T*N*16 bytes of work area + N*T*8 bytes of input staging (+ tables).
template <int N> struct ConvCfg { static constexpr int T = 16, MINB = 2; };    // N < 256
template <> struct ConvCfg<256>  { static constexpr int T = 8, MINB = 3; };
template <> struct ConvCfg<512>  { static constexpr int T = 8, MINB = 2; };
template <> struct ConvCfg<1024> { static constexpr int T = 4, MINB = 2; };
template <> struct ConvCfg<2048> { static constexpr int T = 4, MINB = 1; };
template <> struct ConvCfg<4096> { static constexpr int T = 2, MINB = 1; };

// Persistent grids: number of CTAs that are resident at once (SMs x CTAs per SM), found once per
// kernel instance when the plan sets the shared-memory attribute.
static inline int resident_ctas(const void *kern, int threads, size_t smem) {
    int dev = 0, sms = 0, per_sm = 0;
    cudaGetDevice(&dev);
    cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
    if (cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, kern, threads, smem) != cudaSuccess || per_sm < 1) per_sm = 1;
    return sms * per_sm;
}

template <int N, int MODE>
static cudaError_t launch_col_t(const ColArgs &a, int n_outer, cudaStream_t st, bool set_attr) {
    using C = ColCfg<N>;
    constexpr size_t smem = (size_t)N * C::T * sizeof(float2) * (MODE == MODE_INV ? 2 : 3);
    auto kern = k_col<N, C::T, C::NT, MODE>;
    static int cap = 0;
    if (set_attr) {
        cudaError_t e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
        if (e == cudaSuccess) cap = resident_ctas((const void *)kern, C::NT, smem);
        return e;
    }
    ColArgs b = a;
    b.n_outer = n_outer;
    const long long total = (long long)n_outer * (a.inner_len / C::T);
    const unsigned grid = (unsigned)(total < cap ? total : cap);
    kern<<<grid, C::NT, smem, st>>>(b);
    return cudaGetLastError();
}

// Tensor map of the array k_conv reads: a 2-D tensor of 8-byte elements, dim0 = all columns (x, or
// (ky, kx) in the 3-D z pass), dim1 = the N positions along the line; box = T columns x min(N, 256) rows,
// hardware swizzle matched to the 16-byte-chunk XOR of the staging layout.
typedef CUresult (*tbs_encode_tiled_fn)(CUtensorMap *, CUtensorMapDataType, cuuint32_t, void *, const cuuint64_t *,
                                        const cuuint64_t *, const cuuint32_t *, const cuuint32_t *,
                                        CUtensorMapInterleave, CUtensorMapSwizzle, CUtensorMapL2promotion,
                                        CUtensorMapFloatOOBfill);
static inline cudaError_t make_conv_tensor_map(CUtensorMap *out, const void *base, long long n_cols, int n_rows,
                                               long long row_stride_elems, int T) {
    static tbs_encode_tiled_fn enc = nullptr;
    if (!enc) {
        void *fn = nullptr;
        cudaDriverEntryPointQueryResult q;
        cudaError_t e = cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &fn, cudaEnableDefault, &q);
        if (e != cudaSuccess) return e;
        if (q != cudaDriverEntryPointSuccess || !fn) return cudaErrorNotSupported;
        enc = (tbs_encode_tiled_fn)fn;
    }
    const cuuint64_t dims[2] = {(cuuint64_t)n_cols, (cuuint64_t)n_rows};
    const cuuint64_t strides[1] = {(cuuint64_t)row_stride_elems * 8};
    const cuuint32_t box[2] = {(cuuint32_t)T, (cuuint32_t)(n_rows < 256 ? n_rows : 256)};
    const cuuint32_t estr[2] = {1, 1};
    const CUtensorMapSwizzle sw = T >= 16 ? CU_TENSOR_MAP_SWIZZLE_128B
                                 : T == 8 ? CU_TENSOR_MAP_SWIZZLE_64B
                                 : T == 4 ? CU_TENSOR_MAP_SWIZZLE_32B : CU_TENSOR_MAP_SWIZZLE_NONE;
    const CUresult r = enc(out, CU_TENSOR_MAP_DATA_TYPE_UINT64, 2, const_cast<void *>(base), dims, strides, box, estr,
                           CU_TENSOR_MAP_INTERLEAVE_NONE, sw, CU_TENSOR_MAP_L2_PROMOTION_L2_128B,
                           CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
    return r == CUDA_SUCCESS ? cudaSuccess : cudaErrorInvalidValue;
}
static inline int conv_tile_width(int N);

template <int N, bool KABS>
static cudaError_t launch_conv_tt(const ColArgs &a, const CUtensorMap *tmap, int n_outer, cudaStream_t st, bool set_attr) {
    constexpr int T = ConvCfg<N>::T;
    constexpr int NT = T * tpl_of(N);
    constexpr size_t smem = (size_t)conv_smem_bytes(N, T);
    auto kern = k_conv<N, T, ConvCfg<N>::MINB, KABS>;
    static int cap = 0;
    if (set_attr) {
        cudaError_t e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
        if (e == cudaSuccess) cap = resident_ctas((const void *)kern, NT, smem);
        return e;
    }
    ColArgs b = a;
    b.n_outer = n_outer;
    const long long total = (long long)n_outer * (a.inner_len / T);
    kern<<<(unsigned)(total < cap ? total : cap), NT, smem, st>>>(b, *tmap);
    return cudaGetLastError();
}

template <int N>
static cudaError_t launch_conv_t(const ColArgs &a, const CUtensorMap *tmap, int n_outer, cudaStream_t st, bool set_attr) {
    if (set_attr) {
        cudaError_t e = launch_conv_tt<N, false>(a, tmap, n_outer, st, true);
        return e != cudaSuccess ? e : launch_conv_tt<N, true>(a, tmap, n_outer, st, true);
    }
    return a.kabs.nu > 0.f || a.masked ? launch_conv_tt<N, true>(a, tmap, n_outer, st, false)
                           : launch_conv_tt<N, false>(a, tmap, n_outer, st, false);
}

static cudaError_t launch_conv(int N, const ColArgs &a, const CUtensorMap *tmap, int n_outer, cudaStream_t st,
                               bool set_attr = false) {
    switch (N) {
        case 32:   return launch_conv_t<32>(a, tmap, n_outer, st, set_attr);
        case 64:   return launch_conv_t<64>(a, tmap, n_outer, st, set_attr);
        case 128:  return launch_conv_t<128>(a, tmap, n_outer, st, set_attr);
        case 256:  return launch_conv_t<256>(a, tmap, n_outer, st, set_attr);
        case 512:  return launch_conv_t<512>(a, tmap, n_outer, st, set_attr);
        case 1024: return launch_conv_t<1024>(a, tmap, n_outer, st, set_attr);
        case 2048: return launch_conv_t<2048>(a, tmap, n_outer, st, set_attr);
        case 4096: return launch_conv_t<4096>(a, tmap, n_outer, st, set_attr);
        default: break;
    }
    return cudaErrorInvalidValue;
}
static inline int conv_tile_width(int N) {
    switch (N) {
        case 32: return ConvCfg<32>::T;     case 64: return ConvCfg<64>::T;     case 128: return ConvCfg<128>::T;
        case 256: return ConvCfg<256>::T;   case 512: return ConvCfg<512>::T;   case 1024: return ConvCfg<1024>::T;
        case 2048: return ConvCfg<2048>::T; default: return ConvCfg<4096>::T;
    }
}

template <int MODE>
static cudaError_t launch_col(int N, const ColArgs &a, int n_outer, cudaStream_t st, bool set_attr = false) {
    switch (N) {
        case 32:   return launch_col_t<32, MODE>(a, n_outer, st, set_attr);
        case 64:   return launch_col_t<64, MODE>(a, n_outer, st, set_attr);
        case 128:  return launch_col_t<128, MODE>(a, n_outer, st, set_attr);
        case 256:  return launch_col_t<256, MODE>(a, n_outer, st, set_attr);
        case 512:  return launch_col_t<512, MODE>(a, n_outer, st, set_attr);
        default: break;
    }
    return cudaErrorInvalidValue;
}

template <int N, bool FIRST, bool GEN>
static cudaError_t launch_row_tt(const RowArgs &a, cudaStream_t st, bool set_attr) {
    using C = RowCfg<N>;
    constexpr int TPL = row_tpl_of(N);
    constexpr int GR = TPL >= 32 ? 1 : 32 / TPL;
    constexpr int NT = C::GROUPS * TPL * GR;
    constexpr int ROWS = C::GROUPS * GR;
    constexpr size_t smem = 2 * (size_t)ROWS * LineLay<N>::PITCH * sizeof(float2) +
                            (FIRST || !row_staged(N) ? 0 : (size_t)ROWS * N * sizeof(float4));
    auto kern = k_row<N, C::GROUPS, C::MINB, FIRST, GEN>;
    static int cap = 0;
    if (set_attr) {
        cudaError_t e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
        if (e == cudaSuccess) cap = resident_ctas((const void *)kern, NT, smem);
        return e;
    }
    const int tiles = (a.rows / GR + C::GROUPS - 1) / C::GROUPS;
    kern<<<(unsigned)(tiles < cap ? tiles : cap), NT, smem, st>>>(a);
    return cudaGetLastError();
}

template <int N, bool FIRST>
static cudaError_t launch_row_t(const RowArgs &a, cudaStream_t st, bool set_attr) {
    if (FIRST) return launch_row_tt<N, true, false>(a, st, set_attr);
    if (set_attr) {
        cudaError_t e = launch_row_tt<N, false, false>(a, st, true);
        return e != cudaSuccess ? e : launch_row_tt<N, false, true>(a, st, true);
    }
    return (a.ucbs || a.crit_row >= 0) ? launch_row_tt<N, false, true>(a, st, false)
                                        : launch_row_tt<N, false, false>(a, st, false);
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
