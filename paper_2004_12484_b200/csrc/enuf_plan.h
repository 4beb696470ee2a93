// Internal plan structure and per-precision launch entry points (not part of the C ABI).
#pragma once

#include <cuda_runtime.h>
#include <stdint.h>

#include "enuf_common.cuh"

struct enuf_plan {
    // problem
    int64_t N_cap = 0, N = 0;
    double L = 0, alpha = 0, sigma = 0;   // L = Lb[0]
    double Lb[3] = {0, 0, 0};             // box edges (enuf_plan_create: three times L)
    bool box = false;                     // edges differ: orthorhombic plan (enuf_plan_create_box, R26)
    int k_cut = 0, M = 0, n = 0, m = 0;
    bool mixed = false;                   // n = 3 * 2^k (sigma_s = 1.5): the plain mixed-radix FFT path (enuf_fft_mixed.cuh)
    // options
    int precision = ENUF_F32, window = ENUF_WINDOW_KAISER_BESSEL, variant = ENUF_FORCE_ANALYTIC;
    double lambda = 0.0;
    bool profile = false, keep_spectrum = false;
    bool pdl = true;               // ENUF_OPT_PDL: programmatic dependent launch of the hot-path kernels
    bool trim = false;             // fp32 Kaiser-Bessel m >= 5: kernels visit 2m stencil points per dimension
    cudaStream_t stream = nullptr;
    // ENUF_OPT_CUDA_GRAPH: one evaluation's launches, captured on cap_stream, replayed on `stream`
    bool use_graph = false;
    cudaGraphExec_t gexec = nullptr;
    cudaStream_t cap_stream = nullptr;
    const void* g_r = nullptr; const void* g_q = nullptr; void* g_F = nullptr;   // what the graph was captured for
    int64_t g_N = -1;
    int g_launches = 0;
    // derived
    enuf::TileGeom tg{};
    enuf::WindowParams wp{};
    int Kxp = 0, Ky = 0;
    bool allocated = false, tables_dirty = true, evaluated = false;
    bool bin_count_clean = false;  // bin_count is all zero (left so by the last scan)
    bool real_count_clean = false; // same for real_count
    bool partial_ready = false;    // enuf_spectrum_partial has run and enuf_forces_from_spectrum has not yet
    size_t esize = 4;              // bytes per real
    size_t workspace_bytes = 0;
    int launches = 0;
    cudaError_t launch_error = cudaSuccess;   // error of the last failed kernel launch (launch_ok, enuf_launch.cuh)
    bool q_stage_valid = false;    // the host-API staging buffer holds the charges of the previous host call
    int num_sms = 148;             // multiProcessorCount of the current device (persistent FFT grids)
    // device workspace
    void* rec = nullptr;           // PSlot<T>[N_cap]: record, packed cell, caller index (bin order)
    void* rows = nullptr;          // T[N_cap][3][16]: window rows of the spreading kernel (bin order)
    uint32_t* bin_count = nullptr;    // [nbins]
    uint32_t* bin_offset = nullptr;   // [nbins+1]
    uint32_t* bin_cursor = nullptr;   // [nbins]
    uint2* binrank = nullptr;         // [N_cap] (bin, rank inside the bin) of every particle, from the count pass
    uint32_t* scan_total = nullptr;   // [ceil(nbins / kScanChunk)]
    unsigned long long* scan_desc = nullptr;   // [ceil(nbins / kScanChunk)] (epoch << 32 | chunk total), single-launch scan
    uint32_t* scan_epoch = nullptr;            // [1] device word: evaluation counter, the epoch of scan_desc
    float poly_c[enuf::kPolyMaxDeg + 1][enuf::kMaxM + 1] = {};   // host copy of the polynomial window table
    float poly_d[enuf::kPolyMaxDeg][enuf::kMaxM + 1] = {};       // (fp32 path; packed into PolyArg<m> per launch)
    float bs_c[2 * enuf::kMaxM][2 * enuf::kMaxM + 1] = {};       // B-spline window: exact pieces on d0 in [0, 1/2] (PolyArg::bc, bd)
    float bs_d[2 * enuf::kMaxM][2 * enuf::kMaxM + 1] = {};
    int zchunk = 0;                   // ENUF_OPT_SPREAD_ZCHUNK: fixed pieces of that many planes per spreading CTA (else equal ranges)
    bool zchunk_user = false;
    enuf::SpreadSplit split{};        // work decomposition of the spreading kernel, set per evaluation by launch_bin
    int spread_npx = 4;               // spread column = 8 spread_npx x 16 cells (4 for n >= 128, 2 below)
    int spread_sparse_user = -1;      // ENUF_OPT_SPREAD_SPARSE: -1 auto, 0 / 1 forced
    bool spread_sparse = false;       // fp32: eight-stage ring of 32-slot rounds (few particles per slab and column)
    void* grid[3] = {nullptr, nullptr, nullptr};   // real n^3 (1 for analytic, 3 for ik)
    void* A1[3] = {nullptr, nullptr, nullptr};     // complex [n][n][Kxp]
    void* A2[3] = {nullptr, nullptr, nullptr};     // complex [n][Ky][Kxp]
    void* spectrum = nullptr;      // complex [Ky][Ky][Kxp] (optional)
    void* tw = nullptr;            // complex [n]
    void* iphi = nullptr;          // real [k_cut+1]
    void* wf = nullptr;            // real [k_cut^2+1]
    double* e_partial = nullptr;   // [z-pass CTAs]
    int n_partial = 0;
    double* e_dev = nullptr;       // [1]
    unsigned* fft_done = nullptr;  // [1] CTAs of the Z pass that have published their energy partial
    double* e_pinned = nullptr;    // [1] host
    // real-space part (enuf_real_space; allocated at its first call)
    void* real_pos = nullptr;         // Vec4<T>[N_cap]: wrapped position + charge, cell order
    uint32_t* real_idx = nullptr;     // [N_cap] caller index
    uint32_t* real_count = nullptr;   // [real_ncells]
    uint32_t* real_offset = nullptr;  // [real_ncells + 1]
    uint32_t* real_cursor = nullptr;  // [real_ncells]
    uint32_t* real_scan_total = nullptr;
    double* real_partial = nullptr;   // [2 * ceil(N_cap / 128)]
    double* real_e_dev = nullptr;     // [2] E_real, E_self
    double* real_e_pinned = nullptr;  // [2] host
    int real_ncells_cap = 0;          // cells the count/offset/cursor buffers hold
    int real_ncd = 0, real_s = 0;     // geometry of the last call
    float erfc_c[16] = {};            // fp32 erfc fit of the pair term (enuf_real.cuh, ErfcFit), for x <= erfc_xmax
    float erfc_ua = 0.f, erfc_ub = 0.f;
    double erfc_xmax = -1.0;
    void* r_stage = nullptr;       // host-API staging: r, q, F
    void* q_stage = nullptr;
    void* F_stage = nullptr;
    // profiling: ring of kProfRing evaluations x (ENUF_NUM_STAGES + 1) events
    static constexpr int kMixedScaleCtas = 1024;   // CTAs (= energy partials) of the mixed-radix path's scaling kernel
    static constexpr int kProfRing = 128;
    static constexpr int kProfEv = ENUF_NUM_STAGES + 1;
    cudaEvent_t* ev_ring = nullptr;     // [kProfRing * kProfEv]
    cudaEvent_t* ev = nullptr;          // slot of the current / last evaluation
    int64_t prof_evals = 0;             // evaluations recorded since profiling was switched on
    bool events_valid = false;
};

namespace enuf {

// Implemented once per precision in enuf_kernels_f32.cu / enuf_kernels_f64.cu.
// Each returns the number of kernel launches it issued, or -1 with the CUDA error stored
// in plan->launch_error.
template <typename T> int launch_bin(enuf_plan* p, const void* r, const void* q, void* F);
template <typename T> int launch_spread(enuf_plan* p);
template <typename T> int launch_fft(enuf_plan* p);            // = forward + backward
template <typename T> int launch_fft_forward(enuf_plan* p);    // X, Y forward passes -> A2[0] (partial spectrum)
template <typename T> int launch_fft_backward(enuf_plan* p);   // Z fused + inverse passes + energy
template <typename T> int launch_gather(enuf_plan* p, void* F);
template <typename T> int configure_kernels(enuf_plan* p);   // opt-in shared memory sizes
template <typename T> int spread_ctas_per_sm(int npx);       // resident spreading CTAs per SM
// real-space part: cell sort + pair kernel + energy reduction (enuf_real.cuh)
template <typename T> int launch_real(enuf_plan* p, const void* r, const void* q, double r_cut, int accumulate, void* F);

}  // namespace enuf
