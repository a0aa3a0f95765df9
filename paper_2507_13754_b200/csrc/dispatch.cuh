// dispatch.cuh -- launch configurations per transform length and run-time dispatch.
//
// The kernels of one transform length live in their own translation unit (inst.cu compiled with -DTBS_N=...,
// paper_2507_13754_b200/build.py), so the eight lengths compile in parallel.  This header declares the
// per-length entry points (defined by explicit instantiation in dispatch_impl.cuh / inst.cu) and holds the
// run-time switches over N that tbs.cu calls.
#pragma once
#include "kernels.cuh"

namespace tbs {

// Column-tile kernel k_col (3-D y passes): T adjacent lines per CTA, NT threads.  Shared memory =
// 2*N*T*8 bytes (both parity halves of the padded line) + N*T*8 bytes of input staging (FWD).
template <int N> struct ColCfg { static constexpr int T = 16, NT = 64; };   // N = 32 (and the unused N > 512)
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

// Per-length entry points.  set_attr = true: set the shared-memory attribute of every kernel instance of this
// length and find its persistent grid (number of CTAs resident at once); nothing is launched.
//   launch_row_n : first = true: term 0 forward half (k_row<FIRST>); else the fused inverse+forward k_row (the
//                  general variant when a.ucbs or a.crit_row >= 0 asks for it)
//   launch_conv_n: k_conv (general variant for the k-space potential / masked periodic tables)
//   launch_col_n : k_col, mode = MODE_FWD or MODE_INV (3-D y passes; lengths <= 512)
// LaunchOpt: sm_limit > 0 caps the persistent grid to that many SMs' worth of CTAs (frequency batch: members share
// the GPU); overlap: programmatic dependent launch -- the kernel may be scheduled while its predecessor in the
// stream drains (every kernel waits with griddepcontrol.wait before it touches memory).
struct LaunchOpt {
    int sm_limit = 0;
    bool overlap = false;
};
template <int N> cudaError_t launch_row_n(bool first, const RowArgs &a, cudaStream_t st, bool set_attr, LaunchOpt opt);
template <int N> cudaError_t launch_conv_n(const ColArgs &a, const CUtensorMap *tmap, int n_outer, cudaStream_t st,
                                           bool set_attr, LaunchOpt opt);
template <int N> cudaError_t launch_col_n(int mode, const ColArgs &a, int n_outer, cudaStream_t st, bool set_attr,
                                          LaunchOpt opt);

#define TBS_FOR_EACH_N(X) X(32) X(64) X(128) X(256) X(512) X(1024) X(2048) X(4096)

// Every length is instantiated explicitly in its own translation unit (inst.cu): keep the switches below from
// instantiating all of them wherever the definitions of dispatch_impl.cuh are visible.
#define X(n)                                                                                                          \
    extern template cudaError_t launch_row_n<n>(bool, const RowArgs &, cudaStream_t, bool, LaunchOpt);                       \
    extern template cudaError_t launch_conv_n<n>(const ColArgs &, const CUtensorMap *, int, cudaStream_t, bool, LaunchOpt); \
    extern template cudaError_t launch_col_n<n>(int, const ColArgs &, int, cudaStream_t, bool, LaunchOpt);
TBS_FOR_EACH_N(X)
#undef X

static inline cudaError_t launch_row(int N, bool first, const RowArgs &a, cudaStream_t st, bool set_attr = false,
                                     LaunchOpt opt = LaunchOpt()) {
    switch (N) {
#define X(n) case n: return launch_row_n<n>(first, a, st, set_attr, opt);
        TBS_FOR_EACH_N(X)
#undef X
        default: break;
    }
    return cudaErrorInvalidValue;
}

static inline cudaError_t launch_conv(int N, const ColArgs &a, const CUtensorMap *tmap, int n_outer, cudaStream_t st,
                                      bool set_attr = false, LaunchOpt opt = LaunchOpt()) {
    switch (N) {
#define X(n) case n: return launch_conv_n<n>(a, tmap, n_outer, st, set_attr, opt);
        TBS_FOR_EACH_N(X)
#undef X
        default: break;
    }
    return cudaErrorInvalidValue;
}

static inline cudaError_t launch_col(int N, int mode, const ColArgs &a, int n_outer, cudaStream_t st,
                                     bool set_attr = false, LaunchOpt opt = LaunchOpt()) {
    switch (N) {
        case 32:   return launch_col_n<32>(mode, a, n_outer, st, set_attr, opt);
        case 64:   return launch_col_n<64>(mode, a, n_outer, st, set_attr, opt);
        case 128:  return launch_col_n<128>(mode, a, n_outer, st, set_attr, opt);
        case 256:  return launch_col_n<256>(mode, a, n_outer, st, set_attr, opt);
        case 512:  return launch_col_n<512>(mode, a, n_outer, st, set_attr, opt);
        default: break;
    }
    return cudaErrorInvalidValue;
}

static inline int conv_tile_width(int N) {
    switch (N) {
#define X(n) case n: return ConvCfg<n>::T;
        TBS_FOR_EACH_N(X)
#undef X
        default: break;
    }
    return 0;
}

static inline void radices_of(int N, int &r1, int &r2, int &rl) {
    r1 = r2 = rl = 0;
    switch (N) {
#define X(n) case n: r1 = Radix<n>::R1; r2 = Radix<n>::R2; rl = Radix<n>::RL; break;
        TBS_FOR_EACH_N(X)
#undef X
        default: break;
    }
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

}  // namespace tbs
