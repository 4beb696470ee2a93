// Kernel dispatch for one precision T (included by enuf_kernels_f32.cu / _f64.cu).
#pragma once

#include <type_traits>

#include "enuf_bin.cuh"
#include "enuf_fft.cuh"
#include "enuf_plan.h"
#include "enuf_spread.cuh"

namespace enuf {

template <int V> using IntC = std::integral_constant<int, V>;

// f(IntC<m>, IntC<tile>) -> int
template <typename F>
static inline int dispatch_mt(const enuf_plan* p, F&& f) {
#define ENUF_CASE_M(mv) case mv: return p->tg.T == 16 ? f(IntC<mv>{}, IntC<16>{}) : f(IntC<mv>{}, IntC<8>{});
    switch (p->m) {
        ENUF_CASE_M(1) ENUF_CASE_M(2) ENUF_CASE_M(3) ENUF_CASE_M(4) ENUF_CASE_M(5) ENUF_CASE_M(6)
        default: return -1;
    }
#undef ENUF_CASE_M
}

// f(IntC<n>) -> int
template <typename F>
static inline int dispatch_n(int n, F&& f) {
    switch (n) {
        case 32: return f(IntC<32>{});
        case 64: return f(IntC<64>{});
        case 128: return f(IntC<128>{});
        case 256: return f(IntC<256>{});
        default: return -1;
    }
}

template <typename K>
static inline bool set_smem(K kernel, size_t bytes) {
    return cudaFuncSetAttribute(kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)bytes) == cudaSuccess;
}

template <typename T>
int configure_kernels(enuf_plan* p) {
    int rc = dispatch_mt(p, [&](auto mc, auto tc) -> int {
        constexpr int M_ = decltype(mc)::value, TL = decltype(tc)::value;
        bool ok = set_smem(spread_kernel<T, M_, TL>, spread_smem_bytes<T, M_, TL>());
        ok = ok && set_smem(gather_kernel<T, M_, TL, false>, gather_smem_bytes<T, M_, TL>());
        ok = ok && set_smem(gather_kernel<T, M_, TL, true>, gather_smem_bytes<T, M_, TL>());
        return ok ? 0 : -1;
    });
    if (rc) return rc;
    return dispatch_n(p->n, [&](auto nc) -> int {
        constexpr int N_ = decltype(nc)::value;
        const size_t sb = fft_smem_bytes<T, N_>();
        bool ok = set_smem(fft_x_forward_kernel<T, N_>, sb) && set_smem(fft_x_inverse_kernel<T, N_>, sb)
                  && set_smem(fft_y_forward_kernel<T, N_>, sb) && set_smem(fft_y_inverse_kernel<T, N_>, sb)
                  && set_smem(fft_z_fused_kernel<T, N_, 1>, sb) && set_smem(fft_z_fused_kernel<T, N_, 3>, sb);
        return ok ? 0 : -1;
    });
}

template <typename T>
int launch_bin(enuf_plan* p, const void* r, const void* q, void* F) {
    cudaStream_t s = p->stream;
    const int64_t N = p->N;
    if (cudaMemsetAsync(p->tile_count, 0, sizeof(uint32_t) * p->tg.ntiles, s) != cudaSuccess) return -1;
    const unsigned blocks = (unsigned)((N + 255) / 256);
    bin_count_kernel<T><<<blocks, 256, 0, s>>>(static_cast<const T*>(r), static_cast<const T*>(q),
                                               static_cast<T*>(F), N, p->L, p->tg, p->tile_count);
    bin_scan_kernel<<<1, 1024, 0, s>>>(p->tile_count, p->tile_offset, p->tile_cursor, p->tg.ntiles);
    bin_scatter_kernel<T><<<blocks, 256, 0, s>>>(static_cast<const T*>(r), static_cast<const T*>(q), N, p->L,
                                                 p->tg, p->tile_offset, p->tile_cursor,
                                                 static_cast<PRec<T>*>(p->rec), p->cell, p->idx);
    return cudaGetLastError() == cudaSuccess ? 3 : -1;
}

template <typename T>
int launch_spread(enuf_plan* p) {
    cudaStream_t s = p->stream;
    const size_t n3 = (size_t)p->n * p->n * p->n;
    if (cudaMemsetAsync(p->grid[0], 0, sizeof(T) * n3, s) != cudaSuccess) return -1;
    int rc = dispatch_mt(p, [&](auto mc, auto tc) -> int {
        constexpr int M_ = decltype(mc)::value, TL = decltype(tc)::value;
        using C = TileCfg<M_, TL>;
        spread_kernel<T, M_, TL><<<p->tg.ntiles, C::SPREAD_THREADS, spread_smem_bytes<T, M_, TL>(), s>>>(
            static_cast<const PRec<T>*>(p->rec), p->cell, p->tile_offset, p->tg, p->wp,
            static_cast<T*>(p->grid[0]));
        return 0;
    });
    if (rc) return -1;
    return cudaGetLastError() == cudaSuccess ? 1 : -1;
}

template <typename T>
int launch_fft(enuf_plan* p) {
    cudaStream_t s = p->stream;
    FftGeom fg{p->n, p->k_cut, p->Kxp, p->Ky};
    const Cx<T>* tw = static_cast<const Cx<T>*>(p->tw);
    ScaleTables st{p->iphi, p->wf};
    const int nout = p->variant == ENUF_FORCE_IK ? 3 : 1;
    int launches = dispatch_n(p->n, [&](auto nc) -> int {
        constexpr int N_ = decltype(nc)::value;
        int launches = 0;
        constexpr int LPC = fft_lines_per_cta<N_>();
        const size_t sb = fft_smem_bytes<T, N_>();
        const unsigned bx = (unsigned)(((size_t)N_ * N_) / LPC);
        const unsigned by = (unsigned)(((size_t)N_ * p->Kxp + LPC - 1) / LPC);
        const unsigned bz = (unsigned)(((size_t)p->Ky * p->Kxp + LPC - 1) / LPC);
        if ((int)bz > p->n_partial) return -1;
        fft_x_forward_kernel<T, N_><<<bx, kFftThreads, sb, s>>>(static_cast<const T*>(p->grid[0]),
                                                               static_cast<Cx<T>*>(p->A1[0]), fg, tw);
        fft_y_forward_kernel<T, N_><<<by, kFftThreads, sb, s>>>(static_cast<const Cx<T>*>(p->A1[0]),
                                                               static_cast<Cx<T>*>(p->A2[0]), fg, tw);
        Cx<T>* spec = p->keep_spectrum ? static_cast<Cx<T>*>(p->spectrum) : nullptr;
        if (nout == 1)
            fft_z_fused_kernel<T, N_, 1><<<bz, kFftThreads, sb, s>>>(static_cast<Cx<T>*>(p->A2[0]), nullptr, nullptr,
                                                                    fg, tw, st, p->e_partial, spec);
        else
            fft_z_fused_kernel<T, N_, 3><<<bz, kFftThreads, sb, s>>>(static_cast<Cx<T>*>(p->A2[0]),
                                                                    static_cast<Cx<T>*>(p->A2[1]),
                                                                    static_cast<Cx<T>*>(p->A2[2]), fg, tw, st,
                                                                    p->e_partial, spec);
        launches = 3;
        for (int d = 0; d < nout; ++d) {
            fft_y_inverse_kernel<T, N_><<<by, kFftThreads, sb, s>>>(static_cast<const Cx<T>*>(p->A2[d]),
                                                                   static_cast<Cx<T>*>(p->A1[d]), fg, tw);
            fft_x_inverse_kernel<T, N_><<<bx, kFftThreads, sb, s>>>(static_cast<const Cx<T>*>(p->A1[d]),
                                                                   static_cast<T*>(p->grid[d]), fg, tw);
            launches += 2;
        }
        energy_finish_kernel<<<1, 256, 0, s>>>(p->e_partial, (int)bz, 1.0 / (2.0 * 3.14159265358979323846 * p->L),
                                              p->e_dev);
        launches += 1;
        return launches;
    });
    if (launches < 0) return -1;
    return cudaGetLastError() == cudaSuccess ? launches : -1;
}

template <typename T>
int launch_gather(enuf_plan* p, void* F) {
    cudaStream_t s = p->stream;
    const double PI = 3.14159265358979323846;
    int launches = dispatch_mt(p, [&](auto mc, auto tc) -> int {
        constexpr int M_ = decltype(mc)::value, TL = decltype(tc)::value;
        int launches = 0;
        using C = TileCfg<M_, TL>;
        const size_t sb = gather_smem_bytes<T, M_, TL>();
        if (p->variant == ENUF_FORCE_ANALYTIC) {
            const T pre = (T)(-(double)p->n / (PI * p->L * p->L));
            gather_kernel<T, M_, TL, false><<<p->tg.ntiles, C::GATHER_WARPS * 32, sb, s>>>(
                static_cast<const T*>(p->grid[0]), static_cast<const PRec<T>*>(p->rec), p->cell, p->idx,
                p->tile_offset, p->tg, p->wp, pre, 0, static_cast<T*>(F));
            launches = 1;
        } else {
            const T pre = (T)(2.0 / (p->L * p->L));
            for (int d = 0; d < 3; ++d)
                gather_kernel<T, M_, TL, true><<<p->tg.ntiles, C::GATHER_WARPS * 32, sb, s>>>(
                    static_cast<const T*>(p->grid[d]), static_cast<const PRec<T>*>(p->rec), p->cell, p->idx,
                    p->tile_offset, p->tg, p->wp, pre, d, static_cast<T*>(F));
            launches = 3;
        }
        return launches;
    });
    if (launches < 0) return -1;
    return cudaGetLastError() == cudaSuccess ? launches : -1;
}

}  // namespace enuf
