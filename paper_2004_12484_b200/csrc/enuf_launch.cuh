// Kernel dispatch for one precision T (included by enuf_kernels_f32.cu / _f64.cu).
#pragma once

#include <type_traits>

#include "enuf_bin.cuh"
#include "enuf_fft.cuh"
#include "enuf_fft_mixed.cuh"
#include "enuf_gather.cuh"
#include "enuf_plan.h"
#include "enuf_real.cuh"
#include "enuf_spread.cuh"

namespace enuf {

template <int V> using IntC = std::integral_constant<int, V>;

// f(IntC<m>) -> int
template <typename F>
static inline int dispatch_m(const enuf_plan* p, F&& f) {
    switch (p->m) {
        case 1: return f(IntC<1>{});
        case 2: return f(IntC<2>{});
        case 3: return f(IntC<3>{});
        case 4: return f(IntC<4>{});
        case 5: return f(IntC<5>{});
        case 6: return f(IntC<6>{});
        default: return -1;
    }
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

template <int M_>
static inline PolyArg<M_> make_poly_arg(const enuf_plan* p) {
    PolyArg<M_> a{};
    constexpr int D = PolyArg<M_>::D, NP = PolyArg<M_>::NP;
    static_assert(D % 2 == 0, "packed Horner chains assume an even degree");
    for (int j = 0; j <= M_; ++j) {
        for (int k = 0; k <= D; ++k) a.c[k][j] = p->poly_c[k][j];
        for (int k = 0; k < D; ++k) a.d[k][j] = p->poly_d[k][j];
        a.top[j] = p->poly_c[D][j];
        for (int k = 0; k < NP; ++k) {
            a.vp[k][j] = make_float2(p->poly_c[D - 2 - 2 * k][j], p->poly_c[D - 1 - 2 * k][j]);
            a.dp[k][j] = make_float2(p->poly_d[D - 2 - 2 * k][j], p->poly_d[D - 1 - 2 * k][j]);
        }
    }
    for (int i = 0; i < 2 * M_; ++i)
        for (int jj = 0; jj <= 2 * M_; ++jj) { a.bc[i][jj] = p->bs_c[i][jj]; a.bd[i][jj] = p->bs_d[i][jj]; }
    return a;
}

// After a group of launches: the CUDA error, if any, is taken out of the runtime (cudaGetLastError clears it) and
// kept in the plan, where the C-ABI entry point finds it for enuf_last_error().
static inline bool launch_ok(enuf_plan* p) {
    const cudaError_t e = cudaGetLastError();
    if (e != cudaSuccess) p->launch_error = e;
    return e == cudaSuccess;
}

// Launch with the programmatic-stream-serialization attribute (unless the plan has it switched off): the kernel's CTAs
// may be scheduled while the preceding kernel of the stream still runs and wait in pdl_prologue() (enuf_common.cuh).
template <typename... KArgs, typename... Args>
static inline void pdl_launch(const enuf_plan* p, void (*kernel)(KArgs...), dim3 grid, dim3 block, size_t smem,
                              cudaStream_t s, Args&&... args) {
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = grid; cfg.blockDim = block; cfg.dynamicSmemBytes = smem; cfg.stream = s;
    cudaLaunchAttribute at[1];
    at[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
    at[0].val.programmaticStreamSerializationAllowed = 1;
    cfg.attrs = at; cfg.numAttrs = p->pdl ? 1 : 0;
    (void)cudaLaunchKernelEx(&cfg, kernel, static_cast<KArgs>(args)...);
}

template <typename K>
static inline bool set_smem(K kernel, size_t bytes) {
    return cudaFuncSetAttribute(kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)bytes) == cudaSuccess;
}

// f(IntC<npx>) -> int: patches per column row of the spreading kernel (column = 8 npx x 16 cells)
template <typename F>
static inline int dispatch_npx(int npx, F&& f) {
    return npx == 4 ? f(IntC<4>{}) : f(IntC<2>{});
}

// spread: CTAs the device holds at once for this plan's kernel variant (enuf_spread.cuh)
template <typename T>
int spread_ctas_per_sm(int npx) {
    return npx == 4 ? SpreadCfg<T, 1, false, 4>::CTAS_PER_SM : SpreadCfg<T, 1, false, 2>::CTAS_PER_SM;
}

template <typename T>
int configure_kernels(enuf_plan* p) {
    int rc = dispatch_m(p, [&](auto mc) -> int {
        constexpr int M_ = decltype(mc)::value;
        bool ok = dispatch_npx(p->spread_npx, [&](auto xc) -> int {
            constexpr int NPX = decltype(xc)::value;
            bool k = set_smem(spread_kernel<T, M_, false, NPX>, spread_smem_bytes<T, M_, false, NPX>());
            if constexpr (sizeof(T) == 4)
                k = k && set_smem(spread_kernel<T, M_, false, NPX, true>, spread_smem_bytes<T, M_, false, NPX, true>());
            if constexpr (M_ >= 5 && sizeof(T) == 4) {
                k = k && set_smem(spread_kernel<T, M_, true, NPX>, spread_smem_bytes<T, M_, true, NPX>());
                k = k && set_smem(spread_kernel<T, M_, true, NPX, true>, spread_smem_bytes<T, M_, true, NPX, true>());
            }
            return k ? 0 : -1;
        }) == 0;
        ok = ok && set_smem(gather_kernel<T, M_, false>, gather_smem_bytes<T, M_>());
        ok = ok && set_smem(gather_kernel<T, M_, true>, gather_smem_bytes<T, M_>());
        if constexpr (M_ >= 5 && sizeof(T) == 4) {
            ok = ok && set_smem(gather_kernel<T, M_, false, true>, gather_smem_bytes<T, M_, true>());
            ok = ok && set_smem(gather_kernel<T, M_, true, true>, gather_smem_bytes<T, M_, true>());
        }
        return ok ? 0 : -1;
    });
    if (rc) return rc;
    if (p->mixed) {
        const size_t sb = fft_mixed_smem_bytes<T>(p->n);
        const bool ok = set_smem(fft_mixed_kernel<T, true, false, true>, sb) && set_smem(fft_mixed_kernel<T, false, false, false>, sb)
                        && set_smem(fft_mixed_kernel<T, false, true, true>, sb);
        return ok ? 0 : -1;
    }
    return dispatch_n(p->n, [&](auto nc) -> int {
        constexpr int N_ = decltype(nc)::value;
        const size_t sb = fft_smem_bytes<T, N_>();
        bool ok = set_smem(fft_x_forward_kernel<T, N_>, sb) && set_smem(fft_x_inverse_kernel<T, N_>, sb)
                  && set_smem(fft_x_forward_tma_kernel<T, N_>, fft_xf_tma_smem_bytes<T, N_>())
                  && set_smem(fft_x_inverse_tma_kernel<T, N_>, fft_xi_tma_smem_bytes<T, N_>(p->Kxp))
                  && set_smem(fft_y_forward_kernel<T, N_>, sb) && set_smem(fft_y_inverse_kernel<T, N_>, sb)
                  && set_smem(fft_z_fused_kernel<T, N_, 1>, sb) && set_smem(fft_z_fused_kernel<T, N_, 3>, sb)
                  && set_smem(fft_z_fused_kernel<T, N_, 1, true>, sb) && set_smem(fft_z_fused_kernel<T, N_, 3, true>, sb);
        return ok ? 0 : -1;
    });
}

// Work decomposition of the spreading kernel for this evaluation (SpreadSplit, enuf_common.cuh): equal ranges of slabs,
// as many as the device holds spreading CTAs at once, but none shorter than the planes two pieces share (WZ - 1) + 1;
// ENUF_OPT_SPREAD_ZCHUNK asks for fixed pieces instead.
template <typename T>
static inline SpreadSplit make_spread_split(const enuf_plan* p) {
    return spread_split_make(p->n, p->spread_npx, p->m, p->trim, (long long)p->num_sms * spread_ctas_per_sm<T>(p->spread_npx),
                             p->zchunk_user ? p->zchunk : 0);
}

template <typename T>
int launch_bin(enuf_plan* p, const void* r, const void* q, void* F) {
    cudaStream_t s = p->stream;
    const int64_t N = p->N;
    const int nbins = p->tg.nbins;
    p->split = make_spread_split<T>(p);
    SpreadZero<T> zr{};
    zr.grid = static_cast<T*>(p->grid[0]);
    zr.sp = p->split;
    zr.cx = 8 * p->spread_npx; zr.cy = 16;
    zr.shi = p->trim ? p->m - 1 : p->m;
    zr.nzp = p->split.minlen;
    const unsigned zblocks = (unsigned)(p->split.G + p->split.ncol);
    // the scan clears the histogram behind itself: a memset is needed only when that did not happen
    if (!p->bin_count_clean && cudaMemsetAsync(p->bin_count, 0, sizeof(uint32_t) * nbins, s) != cudaSuccess) return -1;
    p->bin_count_clean = false;
    const unsigned blocks = (unsigned)((N + 255) / 256);
    const unsigned sblocks = (unsigned)((nbins + kScanChunk - 1) / kScanChunk);
    pdl_launch(p, bin_count_kernel<T>, blocks + zblocks, 256, 0, s, static_cast<const T*>(r), static_cast<const T*>(q),
                                               static_cast<T*>(F), N, Edges{{p->Lb[0], p->Lb[1], p->Lb[2]}}, p->tg, p->bin_count, p->scan_epoch, p->binrank,
                                               zblocks, zr);
    int nlaunch = 4;
    if ((int)sblocks <= kScanMaxResident && (int)sblocks <= p->num_sms) {
        // every scan CTA is resident at once: one launch, chunk totals exchanged through scan_desc
        pdl_launch(p, bin_scan_single_kernel, sblocks, kScanThreads, 0, s, p->bin_count, nbins, p->scan_desc, p->scan_epoch,
                                                                p->bin_offset, p->bin_cursor);
        nlaunch = 3;
    } else {
        pdl_launch(p, bin_scan_totals_kernel, sblocks, kScanThreads, 0, s, p->bin_count, nbins, p->scan_total);
        pdl_launch(p, bin_scan_apply_kernel, sblocks, kScanThreads, 0, s, p->bin_count, nbins, p->scan_total, p->bin_offset,
                                                              p->bin_cursor);
    }
    // scatter into bin order and window rows of the sorted particles (read by the spreading kernel).  Small systems: one
    // pass in caller order (one launch less, the slots are not read back).  Large ones: the scatter, then the rows in
    // SORTED order -- 160 B per particle written in one contiguous stream instead of wherever the bins are (measured at
    // N = 1e6: 31 + 36 us for the two against 70 us fused; at N = 1e5: 22.5 against 19.5 us for the whole stage)
    const bool fused = N <= kBinFusedMaxN;
    const unsigned rblocks = (unsigned)((N + 31) / 32);
    const Edges ed{{p->Lb[0], p->Lb[1], p->Lb[2]}};
    if (fused) --nlaunch;                                    // (nlaunch counted the scatter as a launch of its own)
    else pdl_launch(p, bin_scatter_kernel<T>, blocks, 256, 0, s, static_cast<const T*>(r), static_cast<const T*>(q), N,
                    ed, p->tg, p->bin_offset, p->binrank, static_cast<PSlot<T>*>(p->rec));
    const int rc = dispatch_m(p, [&](auto mc) -> int {
        constexpr int M_ = decltype(mc)::value;
        const PolyArg<M_> pa = make_poly_arg<M_>(p);
        auto run = [&](auto trim_c) -> int {
            constexpr bool kTrim = decltype(trim_c)::value != 0;
            if (fused)
                pdl_launch(p, bin_place_kernel<T, M_, kTrim>, rblocks, kRowsThreads, 0, s, static_cast<const T*>(r),
                    static_cast<const T*>(q), N, ed, p->tg, p->bin_offset, p->binrank, static_cast<PSlot<T>*>(p->rec), p->wp, pa,
                    static_cast<T*>(p->rows));
            else
                pdl_launch(p, window_rows_kernel<T, M_, kTrim>, rblocks, kRowsThreads, 0, s,
                    static_cast<const PSlot<T>*>(p->rec), p->bin_offset, nbins, p->wp, pa, static_cast<T*>(p->rows));
            return 0;
        };
        if constexpr (M_ >= 5 && sizeof(T) == 4) {
            if (p->trim) return run(IntC<1>{});
        }
        return run(IntC<0>{});
    });
    if (rc || !launch_ok(p)) return -1;
    ++nlaunch;
    p->bin_count_clean = true;
    return nlaunch;
}

template <typename T>
int launch_spread(enuf_plan* p) {
    cudaStream_t s = p->stream;
    int rc = dispatch_m(p, [&](auto mc) -> int {
        constexpr int M_ = decltype(mc)::value;
        return dispatch_npx(p->spread_npx, [&](auto xc) -> int {
            constexpr int NPX = decltype(xc)::value;
            auto run = [&](auto trim_c) -> int {
                constexpr bool kTrim = decltype(trim_c)::value != 0;
                using C = SpreadCfg<T, M_, kTrim, NPX>;
                const dim3 grid((unsigned)p->split.G);          // set by launch_bin, whose extra blocks cleared the shared planes
                if constexpr (sizeof(T) == 4) {
                    if (p->spread_sparse) {      // few particles per slab: 8 stages of 32 slots (SpreadCfg)
                        pdl_launch(p, spread_kernel<T, M_, kTrim, NPX, true>, grid, C::NT,
                                   spread_smem_bytes<T, M_, kTrim, NPX, true>(), s,
                                   static_cast<const PSlot<T>*>(p->rec), static_cast<const T*>(p->rows), p->bin_offset, p->tg,
                                   p->split, static_cast<T*>(p->grid[0]));
                        return 0;
                    }
                }
                pdl_launch(p, spread_kernel<T, M_, kTrim, NPX>, grid, C::NT, spread_smem_bytes<T, M_, kTrim, NPX>(), s, 
                    static_cast<const PSlot<T>*>(p->rec), static_cast<const T*>(p->rows), p->bin_offset, p->tg,
                    p->split, static_cast<T*>(p->grid[0]));
                return 0;
            };
            if constexpr (M_ >= 5 && sizeof(T) == 4) {
                if (p->trim) return run(IntC<1>{});
            }
            return run(IntC<0>{});
        });
    });
    if (rc) return -1;
    return launch_ok(p) ? 1 : -1;
}

// Forward half of the FFT stage (a3): X real-to-complex and Y passes; leaves the partial spectrum
// [z][ky'][kx] of this plan's particles in A2[0].  Linear in the charges, so partial spectra of
// particle subsets add (Eq. 61): the multi-GPU path all-reduces A2[0] here.
// Grids of 3 * 2^k points (enuf_fft_mixed.cuh): three line-transform launches per 3-D FFT on the full complex grid A1.
template <typename T>
static inline void launch_mixed_pass(enuf_plan* p, int dir, int sign, const void* in, void* out) {
    const size_t n = (size_t)p->n, sb = fft_mixed_smem_bytes<T>(p->n);
    const unsigned blocks = (unsigned)(n * n / mix_lines<T>());
    const Cx<T>* tw = static_cast<const Cx<T>*>(p->tw);
    if (dir == 0 && sign < 0)        // X forward: real grid in
        pdl_launch(p, fft_mixed_kernel<T, true, false, true>, blocks, kFftThreads, sb, p->stream, in, out, p->n, n * n, n, (size_t)1, sign, tw);
    else if (dir == 0)               // X inverse: real grid out
        pdl_launch(p, fft_mixed_kernel<T, false, true, true>, blocks, kFftThreads, sb, p->stream, in, out, p->n, n * n, n, (size_t)1, sign, tw);
    else if (dir == 1)
        pdl_launch(p, fft_mixed_kernel<T, false, false, false>, blocks, kFftThreads, sb, p->stream, in, out, p->n, n * n, (size_t)1, n, sign, tw);
    else
        pdl_launch(p, fft_mixed_kernel<T, false, false, false>, blocks, kFftThreads, sb, p->stream, in, out, p->n, n, (size_t)1, n * n, sign, tw);
}

template <typename T>
int launch_fft_forward(enuf_plan* p) {
    if (p->mixed) {
        launch_mixed_pass<T>(p, 0, -1, p->grid[0], p->A1[0]);
        launch_mixed_pass<T>(p, 1, -1, p->A1[0], p->A1[0]);
        launch_mixed_pass<T>(p, 2, -1, p->A1[0], p->A1[0]);
        return launch_ok(p) ? 3 : -1;
    }
    cudaStream_t s = p->stream;
    FftGeom fg{p->n, p->k_cut, p->Kxp, p->Ky};
    const Cx<T>* tw = static_cast<const Cx<T>*>(p->tw);
    int launches = dispatch_n(p->n, [&](auto nc) -> int {
        constexpr int N_ = decltype(nc)::value;
        constexpr int LPC = fft_lines_per_cta<N_>();
        const size_t sb = fft_smem_bytes<T, N_>();
        const unsigned bx = (unsigned)(((size_t)N_ * N_) / LPC);
        const unsigned by = (unsigned)(((size_t)N_ * p->Kxp + LPC - 1) / LPC);
        {
            // persistent, rows staged through TMA; CTAs per SM by shared memory (<= 3 for fp32, 1-2 for fp64)
            const size_t sbt = fft_xf_tma_smem_bytes<T, N_>();
            const int per_sm = (int)((size_t)(227 * 1024) / (sbt + 1024));
            const int ntiles = (int)(bx / 2);
            const int gridx = ntiles < p->num_sms * per_sm ? ntiles : p->num_sms * per_sm;
            pdl_launch(p, fft_x_forward_tma_kernel<T, N_>, gridx, kFftThreads, sbt, s, static_cast<const T*>(p->grid[0]),
                                                                           static_cast<Cx<T>*>(p->A1[0]), fg, tw, ntiles);
        }
        pdl_launch(p, fft_y_forward_kernel<T, N_>, by, kFftThreads, sb, s, static_cast<const Cx<T>*>(p->A1[0]),
                                                               static_cast<Cx<T>*>(p->A2[0]), fg, tw);
        return 2;
    });
    if (launches < 0) return -1;
    return launch_ok(p) ? launches : -1;
}

// Backward half (a4 + a5 + a7): Z forward . scale . energy . Z inverse on A2[0] (in place; the ik
// variant writes A2[0..2]), Y and X inverse passes into the real field(s), energy reduction.
template <typename T>
int launch_fft_backward(enuf_plan* p) {
    if (p->mixed) {
        const int nout = p->variant == ENUF_FORCE_IK ? 3 : 1;
        const double PI = 3.14159265358979323846;
        ScaleTables st{p->iphi, p->wf};
        Cx<T>* spec = p->keep_spectrum ? static_cast<Cx<T>*>(p->spectrum) : nullptr;
        Cx<T>* c0 = static_cast<Cx<T>*>(p->A1[0]);
        Cx<T>* c1 = nout == 3 ? static_cast<Cx<T>*>(p->A1[1]) : nullptr;
        Cx<T>* c2 = nout == 3 ? static_cast<Cx<T>*>(p->A1[2]) : nullptr;
        // Eq. 38: C/(2 pi L), C = 1; a box (weights in length^2): 1/(2 pi V)
        const double e_scale = p->box ? 1.0 / (2.0 * PI * p->Lb[0] * p->Lb[1] * p->Lb[2]) : 1.0 / (2.0 * PI * p->L);
        BoxScale bs{};
        {
            double lm = p->Lb[0] > p->Lb[1] ? p->Lb[0] : p->Lb[1];
            lm = lm > p->Lb[2] ? lm : p->Lb[2];
            for (int d = 0; d < 3; ++d) { bs.a[d] = (lm / p->Lb[d]) * (lm / p->Lb[d]); bs.l[d] = p->Lb[d]; }
            bs.lm2 = lm * lm; bs.alpha = p->alpha; bs.lambda = p->lambda;
        }
        const unsigned ctas = enuf_plan::kMixedScaleCtas;
        if (nout == 1 && !p->box)
            pdl_launch(p, mixed_scale_kernel<T, 1, false>, ctas, kFftThreads, 0, p->stream, c0, c1, c2, p->n, p->k_cut, p->Kxp,
                       p->Ky, st, p->e_partial, spec, p->fft_done, e_scale, p->e_dev, bs);
        else if (nout == 1)
            pdl_launch(p, mixed_scale_kernel<T, 1, true>, ctas, kFftThreads, 0, p->stream, c0, c1, c2, p->n, p->k_cut, p->Kxp,
                       p->Ky, st, p->e_partial, spec, p->fft_done, e_scale, p->e_dev, bs);
        else if (!p->box)
            pdl_launch(p, mixed_scale_kernel<T, 3, false>, ctas, kFftThreads, 0, p->stream, c0, c1, c2, p->n, p->k_cut, p->Kxp,
                       p->Ky, st, p->e_partial, spec, p->fft_done, e_scale, p->e_dev, bs);
        else
            pdl_launch(p, mixed_scale_kernel<T, 3, true>, ctas, kFftThreads, 0, p->stream, c0, c1, c2, p->n, p->k_cut, p->Kxp,
                       p->Ky, st, p->e_partial, spec, p->fft_done, e_scale, p->e_dev, bs);
        for (int d = 0; d < nout; ++d) {
            launch_mixed_pass<T>(p, 2, +1, p->A1[d], p->A1[d]);
            launch_mixed_pass<T>(p, 1, +1, p->A1[d], p->A1[d]);
            launch_mixed_pass<T>(p, 0, +1, p->A1[d], p->grid[d]);
        }
        return launch_ok(p) ? 1 + 3 * nout : -1;
    }
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
        Cx<T>* spec = p->keep_spectrum ? static_cast<Cx<T>*>(p->spectrum) : nullptr;
        // Eq. 38: C/(2 pi L), C = 1; a box (weights in length^2, fft_z_fused_kernel): 1/(2 pi V)
        const double PI = 3.14159265358979323846;
        const double e_scale = p->box ? 1.0 / (2.0 * PI * p->Lb[0] * p->Lb[1] * p->Lb[2]) : 1.0 / (2.0 * PI * p->L);
        BoxScale bs{};
        {
            double lm = p->Lb[0] > p->Lb[1] ? p->Lb[0] : p->Lb[1];
            lm = lm > p->Lb[2] ? lm : p->Lb[2];
            for (int d = 0; d < 3; ++d) { bs.a[d] = (lm / p->Lb[d]) * (lm / p->Lb[d]); bs.l[d] = p->Lb[d]; }
            bs.lm2 = lm * lm; bs.alpha = p->alpha; bs.lambda = p->lambda;
        }
        Cx<T>* a0 = static_cast<Cx<T>*>(p->A2[0]);
        Cx<T>* a1 = nout == 3 ? static_cast<Cx<T>*>(p->A2[1]) : nullptr;
        Cx<T>* a2 = nout == 3 ? static_cast<Cx<T>*>(p->A2[2]) : nullptr;
        if (nout == 1 && !p->box)
            pdl_launch(p, fft_z_fused_kernel<T, N_, 1>, bz, kFftThreads, sb, s, a0, a1, a2, fg, tw, st, p->e_partial, spec,
                       p->fft_done, e_scale, p->e_dev, bs);
        else if (nout == 1)
            pdl_launch(p, fft_z_fused_kernel<T, N_, 1, true>, bz, kFftThreads, sb, s, a0, a1, a2, fg, tw, st, p->e_partial, spec,
                       p->fft_done, e_scale, p->e_dev, bs);
        else if (!p->box)
            pdl_launch(p, fft_z_fused_kernel<T, N_, 3>, bz, kFftThreads, sb, s, a0, a1, a2, fg, tw, st, p->e_partial, spec,
                       p->fft_done, e_scale, p->e_dev, bs);
        else
            pdl_launch(p, fft_z_fused_kernel<T, N_, 3, true>, bz, kFftThreads, sb, s, a0, a1, a2, fg, tw, st, p->e_partial, spec,
                       p->fft_done, e_scale, p->e_dev, bs);
        launches = 1;
        for (int d = 0; d < nout; ++d) {
            pdl_launch(p, fft_y_inverse_kernel<T, N_>, by, kFftThreads, sb, s, static_cast<const Cx<T>*>(p->A2[d]),
                                                                   static_cast<Cx<T>*>(p->A1[d]), fg, tw);
            {
                const size_t sbt = fft_xi_tma_smem_bytes<T, N_>(p->Kxp);
                const int per_sm = (int)((size_t)(227 * 1024) / (sbt + 1024));
                const int ntiles = (int)(bx / 2);
                const int cap = p->num_sms * (per_sm < 4 ? per_sm : 4);
                pdl_launch(p, fft_x_inverse_tma_kernel<T, N_>, ntiles < cap ? ntiles : cap, kFftThreads, sbt, s, 
                    static_cast<const Cx<T>*>(p->A1[d]), static_cast<T*>(p->grid[d]), fg, tw, ntiles);
            }
            launches += 2;
        }
        return launches;
    });
    if (launches < 0) return -1;
    return launch_ok(p) ? launches : -1;
}

template <typename T>
int launch_fft(enuf_plan* p) {
    const int a = launch_fft_forward<T>(p);
    if (a < 0) return -1;
    const int b = launch_fft_backward<T>(p);
    return b < 0 ? -1 : a + b;
}

template <typename T>
int launch_gather(enuf_plan* p, void* F) {
    cudaStream_t s = p->stream;
    const double PI = 3.14159265358979323846;
    int launches = dispatch_m(p, [&](auto mc) -> int {
        constexpr int M_ = decltype(mc)::value;
        const unsigned ntiles = (unsigned)(p->tg.nt * p->tg.nt * (p->n / kTile));
        const PolyArg<M_> pa = make_poly_arg<M_>(p);
        auto run = [&](auto trim_c) -> int {
            constexpr bool kTrim = decltype(trim_c)::value != 0;
            using C = GatherCfg<M_, kTrim>;
            const size_t sb = gather_smem_bytes<T, M_, kTrim>();
            if (p->variant == ENUF_FORCE_ANALYTIC) {
                // cubic: -n/(pi L^2); box: -n/(pi V L_d), as the x value and the ratios L_x/L_y, L_x/L_z (1 when cubic)
                const double vol = p->Lb[0] * p->Lb[1] * p->Lb[2];
                const T pre = p->box ? (T)(-(double)p->n / (PI * vol * p->Lb[0])) : (T)(-(double)p->n / (PI * p->L * p->L));
                const T ry = p->box ? (T)(p->Lb[0] / p->Lb[1]) : (T)1, rz = p->box ? (T)(p->Lb[0] / p->Lb[2]) : (T)1;
                pdl_launch(p, gather_kernel<T, M_, false, kTrim>, ntiles, C::NT, sb, s, 
                    static_cast<const T*>(p->grid[0]), static_cast<const PSlot<T>*>(p->rec),
                    p->bin_offset, p->tg, p->wp, pa, pre, 0, static_cast<T*>(F), ry, rz);
                return 1;
            }
            // Eq. 42: 2/L^2 with b^_d = -i n_d ..; box: 2/V with b^_d = -i h_d .. (fft_z_fused_kernel)
            const T pre = p->box ? (T)(2.0 / (p->Lb[0] * p->Lb[1] * p->Lb[2])) : (T)(2.0 / (p->L * p->L));
            for (int d = 0; d < 3; ++d)
                pdl_launch(p, gather_kernel<T, M_, true, kTrim>, ntiles, C::NT, sb, s, 
                    static_cast<const T*>(p->grid[d]), static_cast<const PSlot<T>*>(p->rec),
                    p->bin_offset, p->tg, p->wp, pa, pre, d, static_cast<T*>(F), (T)1, (T)1);
            return 3;
        };
        if constexpr (M_ >= 5 && sizeof(T) == 4) {
            if (p->trim) return run(IntC<1>{});
        }
        return run(IntC<0>{});
    });
    if (launches < 0) return -1;
    return launch_ok(p) ? launches : -1;
}

template <typename T>
int launch_real(enuf_plan* p, const void* r, const void* q, double r_cut, int accumulate, void* F) {
    cudaStream_t s = p->stream;
    const int64_t N = p->N;
    const RealGeom g{p->real_ncd, p->real_s, p->L};
    const int ncells = g.ncd * g.ncd * g.ncd;
    using V4 = typename Vec4<T>::type;
    if (!p->real_count_clean && cudaMemsetAsync(p->real_count, 0, sizeof(uint32_t) * ncells, s) != cudaSuccess) return -1;
    p->real_count_clean = false;
    const unsigned blocks = (unsigned)((N + 255) / 256);
    const unsigned sblocks = (unsigned)((ncells + kScanChunk - 1) / kScanChunk);
    real_count_kernel<T><<<blocks, 256, 0, s>>>(static_cast<const T*>(r), static_cast<const T*>(q), static_cast<T*>(F),
                                                accumulate ? 0 : 1, N, g, p->real_count);
    bin_scan_totals_kernel<<<sblocks, kScanThreads, 0, s>>>(p->real_count, ncells, p->real_scan_total);
    bin_scan_apply_kernel<<<sblocks, kScanThreads, 0, s>>>(p->real_count, ncells, p->real_scan_total, p->real_offset,
                                                          p->real_cursor);
    real_scatter_kernel<T><<<blocks, 256, 0, s>>>(static_cast<const T*>(r), static_cast<const T*>(q), N, g,
                                                  p->real_cursor, static_cast<V4*>(p->real_pos), p->real_idx);
    const unsigned fblocks = (unsigned)((N + kRealThreads - 1) / kRealThreads);
    const T alpha = (T)p->alpha, rc2 = (T)(r_cut * r_cut);
    ErfcFit ef;
    for (int k = 0; k <= kErfcDeg; ++k) ef.c[k] = p->erfc_c[k];
    ef.ua = p->erfc_ua; ef.ub = p->erfc_ub;
    if (p->lambda > 0.0)
        real_force_kernel<T, true><<<fblocks, kRealThreads, 0, s>>>(
            static_cast<const V4*>(p->real_pos), p->real_idx, p->real_offset, ncells, g, alpha, rc2,
            (T)(1.0 / p->lambda), ef, accumulate, static_cast<T*>(F), p->real_partial);
    else
        real_force_kernel<T, false><<<fblocks, kRealThreads, 0, s>>>(
            static_cast<const V4*>(p->real_pos), p->real_idx, p->real_offset, ncells, g, alpha, rc2, (T)0,
            ef, accumulate, static_cast<T*>(F), p->real_partial);
    real_energy_finish_kernel<<<1, 256, 0, s>>>(p->real_partial, (int)fblocks, 0.5,
                                               p->alpha * 0.56418958354775628694807945156077, p->real_e_dev);
    if (!launch_ok(p)) return -1;
    p->real_count_clean = true;      // the scan cleared the cell histogram (all real_ncells_cap entries beyond ncells stay 0)
    return 6;
}

}  // namespace enuf
