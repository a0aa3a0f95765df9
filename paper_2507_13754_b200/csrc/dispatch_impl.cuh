// dispatch_impl.cuh -- the launch templates behind the per-length entry points of dispatch.cuh.  Included only by
// inst.cu, which is compiled once per transform length.
#pragma once
#include "dispatch.cuh"

namespace tbs {

// Persistent grids: number of CTAs that are resident at once (SMs x CTAs per SM), found once per
// kernel instance when the plan sets the shared-memory attribute.
struct Resident {
    int sms = 0, per_sm = 0;
    // CTAs of a persistent launch: everything resident, or `sm_limit` SMs' worth
    long long cap(int sm_limit) const { return (long long)per_sm * (sm_limit > 0 && sm_limit < sms ? sm_limit : sms); }
};
static inline Resident resident_ctas(const void *kern, int threads, size_t smem) {
    Resident r;
    int dev = 0;
    cudaGetDevice(&dev);
    cudaDeviceGetAttribute(&r.sms, cudaDevAttrMultiProcessorCount, dev);
    if (cudaOccupancyMaxActiveBlocksPerMultiprocessor(&r.per_sm, kern, threads, smem) != cudaSuccess || r.per_sm < 1) r.per_sm = 1;
    return r;
}

// One launch; overlap = programmatic stream serialization (the kernel's CTAs may become resident while the
// previous kernel of the stream drains; griddepcontrol.wait in the kernel orders the memory accesses).
template <class... KArgs, class... Args>
static cudaError_t launch_k(void (*kern)(KArgs...), unsigned grid, int threads, size_t smem, cudaStream_t st, bool overlap,
                            Args... args) {
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = dim3(grid);
    cfg.blockDim = dim3(threads);
    cfg.dynamicSmemBytes = smem;
    cfg.stream = st;
    cudaLaunchAttribute at[1];
    at[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
    at[0].val.programmaticStreamSerializationAllowed = 1;
    cfg.attrs = at;
    cfg.numAttrs = overlap ? 1 : 0;
    return cudaLaunchKernelEx(&cfg, kern, KArgs(args)...);
}

template <int N, int MODE>
static cudaError_t launch_col_t(const ColArgs &a, int n_outer, cudaStream_t st, bool set_attr, LaunchOpt opt) {
    using C = ColCfg<N>;
    constexpr size_t smem = (size_t)N * C::T * sizeof(float2) * (MODE == MODE_INV ? 2 : 3);
    auto kern = k_col<N, C::T, C::NT, MODE>;
    static Resident res;
    if (set_attr) {
        cudaError_t e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
        if (e == cudaSuccess) res = resident_ctas((const void *)kern, C::NT, smem);
        return e;
    }
    ColArgs b = a;
    b.n_outer = n_outer;
    const long long total = (long long)n_outer * (a.inner_len / C::T);
    const long long cap = res.cap(opt.sm_limit);
    return launch_k(kern, (unsigned)(total < cap ? total : cap), C::NT, smem, st, opt.overlap, b);
}

template <int N, bool KABS, bool PER = false, bool TWOF = false>
static cudaError_t launch_conv_tt(const ColArgs &a, const CUtensorMap *tmap, int n_outer, cudaStream_t st, bool set_attr,
                                  LaunchOpt opt) {
    constexpr int T = ConvCfg<N>::T;
    constexpr int NT = (PER ? T / 2 : T) * tpl_of(N);
    constexpr size_t smem = PER ? (size_t)conv_smem_bytes_per(N, T) : (size_t)conv_smem_bytes(N, T);
    auto kern = k_conv<N, T, ConvCfg<N>::MINB, KABS, PER, TWOF>;
    static Resident res;
    if (set_attr) {
        cudaError_t e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
        if (e == cudaSuccess) res = resident_ctas((const void *)kern, NT, smem);
        return e;
    }
    ColArgs b = a;
    b.n_outer = n_outer;
    const long long total = (long long)n_outer * (a.inner_len / T);
    const long long cap = res.cap(opt.sm_limit);
    return launch_k(kern, (unsigned)(total < cap ? total : cap), NT, smem, st, opt.overlap, b, *tmap);
}

template <int N, bool FIRST, bool GEN, bool PER = false, bool TWOF = false>
static cudaError_t launch_row_tt(const RowArgs &a, cudaStream_t st, bool set_attr, LaunchOpt opt) {
    using C = RowCfg<N>;
    constexpr int TPL = row_tpl_of(N);
    constexpr int GR = TPL >= 32 ? 1 : 32 / TPL;
    constexpr int NT = C::GROUPS * TPL * GR;
    constexpr int ROWS = C::GROUPS * GR;
    constexpr size_t smem = 2 * (size_t)ROWS * LineLay<N>::PITCH * sizeof(float2) +
                            (FIRST || !row_staged(N) ? 0 : (size_t)ROWS * N * sizeof(float4));
    auto kern = k_row<N, C::GROUPS, C::MINB, FIRST, GEN, PER, TWOF>;
    static Resident res;
    if (set_attr) {
        cudaError_t e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
        if (e == cudaSuccess) res = resident_ctas((const void *)kern, NT, smem);
        return e;
    }
    const long long tiles = (a.rows / (GR * (PER ? 2 : 1)) + C::GROUPS - 1) / C::GROUPS;
    const long long cap = res.cap(opt.sm_limit);
    return launch_k(kern, (unsigned)(tiles < cap ? tiles : cap), NT, smem, st, opt.overlap, a);
}

template <int N>
cudaError_t launch_row_n(bool first, const RowArgs &a, cudaStream_t st, bool set_attr, LaunchOpt opt) {
    if (set_attr) {
        cudaError_t e = launch_row_tt<N, true, false>(a, st, true, LaunchOpt());
        if (e == cudaSuccess) e = launch_row_tt<N, false, false>(a, st, true, LaunchOpt());
        if (e == cudaSuccess) e = launch_row_tt<N, false, true>(a, st, true, LaunchOpt());
        if (e == cudaSuccess) e = launch_row_tt<N, true, false, true>(a, st, true, LaunchOpt());
        if (e == cudaSuccess) e = launch_row_tt<N, false, true, true>(a, st, true, LaunchOpt());
        if (e == cudaSuccess) e = launch_row_tt<N, true, false, false, true>(a, st, true, LaunchOpt());
        if (e == cudaSuccess) e = launch_row_tt<N, false, true, false, true>(a, st, true, LaunchOpt());
        return e;
    }
    if (a.per == 2) return first ? launch_row_tt<N, true, false, false, true>(a, st, false, opt)
                                 : launch_row_tt<N, false, true, false, true>(a, st, false, opt);
    if (a.per) return first ? launch_row_tt<N, true, false, true>(a, st, false, opt)
                            : launch_row_tt<N, false, true, true>(a, st, false, opt);
    if (first) return launch_row_tt<N, true, false>(a, st, false, opt);
    return (a.ucbs || a.crit_row >= 0) ? launch_row_tt<N, false, true>(a, st, false, opt)
                                        : launch_row_tt<N, false, false>(a, st, false, opt);
}

template <int N>
cudaError_t launch_conv_n(const ColArgs &a, const CUtensorMap *tmap, int n_outer, cudaStream_t st, bool set_attr,
                          LaunchOpt opt) {
    if (set_attr) {
        cudaError_t e = launch_conv_tt<N, false>(a, tmap, n_outer, st, true, LaunchOpt());
        if (e == cudaSuccess) e = launch_conv_tt<N, true>(a, tmap, n_outer, st, true, LaunchOpt());
        if (e == cudaSuccess) e = launch_conv_tt<N, true, true>(a, tmap, n_outer, st, true, LaunchOpt());
        if (e == cudaSuccess) e = launch_conv_tt<N, true, true, true>(a, tmap, n_outer, st, true, LaunchOpt());
        return e;
    }
    if (a.per == 2) return launch_conv_tt<N, true, true, true>(a, tmap, n_outer, st, false, opt);
    if (a.per) return launch_conv_tt<N, true, true>(a, tmap, n_outer, st, false, opt);
    return a.kabs.nu > 0.f || a.masked ? launch_conv_tt<N, true>(a, tmap, n_outer, st, false, opt)
                                       : launch_conv_tt<N, false>(a, tmap, n_outer, st, false, opt);
}

template <int N>
cudaError_t launch_col_n(int mode, const ColArgs &a, int n_outer, cudaStream_t st, bool set_attr, LaunchOpt opt) {
    if (set_attr) {
        cudaError_t e = launch_col_t<N, MODE_FWD>(a, n_outer, st, true, LaunchOpt());
        return e != cudaSuccess ? e : launch_col_t<N, MODE_INV>(a, n_outer, st, true, LaunchOpt());
    }
    return mode == MODE_FWD ? launch_col_t<N, MODE_FWD>(a, n_outer, st, false, opt)
                            : launch_col_t<N, MODE_INV>(a, n_outer, st, false, opt);
}

}  // namespace tbs
