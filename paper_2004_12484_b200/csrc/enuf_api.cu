// C ABI of libenuf_b200.so (see include/enuf.h): plan life cycle, host-side tables
// (step a0) and the orchestration of one evaluation a1..a7 on the plan's stream.
#include <cmath>
#include <cstdarg>
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <new>
#include <vector>

#include "enuf_plan.h"

namespace {

thread_local char g_err[512] = "";

int fail(int code, const char* fmt, ...) {
    va_list ap;
    va_start(ap, fmt);
    vsnprintf(g_err, sizeof(g_err), fmt, ap);
    va_end(ap);
    return code;
}

int fail_cuda(cudaError_t e, const char* what);
// a launch_* helper returned -1: its CUDA error was stored in the plan (launch_ok, enuf_launch.cuh)
int fail_launch(enuf_plan* p) {
    const cudaError_t e = p->launch_error != cudaSuccess ? p->launch_error : cudaErrorUnknown;
    p->launch_error = cudaSuccess;
    return fail_cuda(e, "kernel launch");
}

int fail_cuda(cudaError_t e, const char* what) {
    snprintf(g_err, sizeof(g_err), "%s: %s", what, cudaGetErrorString(e));
    (void)cudaGetLastError();
    return ENUF_ECUDA;
}

#define CU(call)                                                   \
    do {                                                           \
        cudaError_t e__ = (call);                                  \
        if (e__ != cudaSuccess) return fail_cuda(e__, #call);      \
    } while (0)

constexpr double kPi = 3.14159265358979323846264338327950288;

// modified Bessel function of the first kind, order 0 (power series; x <= ~60 here)
double bessel_i0_series(double x) {
    const double q = 0.25 * x * x;
    double term = 1.0, sum = 1.0;
    for (int k = 1; k < 1000; ++k) {
        term *= q / ((double)k * (double)k);
        sum += term;
        if (term <= 1e-18 * sum) break;
    }
    return sum;
}

// B_p(x) and its i-th derivative from the right, B_p^(i)(x) = sum_l (-1)^l C(i, l) B_{p-i}(x + i/2 - l)
// (B_p' = B_{p-1}(. + 1/2) - B_{p-1}(. - 1/2) applied i times); host, fp64, p <= 12
double bspline_host(int p, double x) {
    const double t = x + 0.5 * p;
    if (!(t >= 0.0) || !(t < p)) return 0.0;
    double a[16] = {0};
    a[(int)t] = 1.0;                                   // right-continuous at the knots
    for (int k = 2; k <= p; ++k)
        for (int j = 0; j + k <= p; ++j) a[j] = ((t - j) * a[j] + (k - t + j) * a[j + 1]) / (k - 1);
    return a[0];
}
double bspline_deriv_host(int p, int i, double x) {
    double s = 0.0, binom = 1.0;
    for (int l = 0; l <= i; ++l) {
        s += ((l & 1) ? -1.0 : 1.0) * binom * bspline_host(p - i, x + 0.5 * i - l);
        binom = binom * (i - l) / (l + 1);
    }
    return s;
}

// Window transform Phi(k) = int phi(d) exp(-2 pi i k d/n) dd for the phi(0)=1 windows (R6, R7)
double window_transform(const enuf_plan* p, int k) {
    const double m = p->m, sg = p->sigma, n = p->n;
    if (p->window == ENUF_WINDOW_SINC_POWER) {
        // sinc(pi c d) is the transform of a box of width c and height 1/c; its 2m-th power that of their 2m-fold convolution
        const double c = (2.0 - 1.0 / sg) / (2.0 * m);
        return bspline_host(2 * p->m, k / (n * c)) / c;
    }
    if (p->window == ENUF_WINDOW_BSPLINE) {
        // the order-2m B-spline is the 2m-fold convolution of the unit box: sinc(pi k/n)^(2m), over B_2m(0)
        const double t = kPi * k / n, sc = k == 0 ? 1.0 : std::sin(t) / t;
        return std::pow(sc, 2 * p->m) / bspline_host(2 * p->m, 0.0);
    }
    if (p->window == ENUF_WINDOW_GAUSSIAN) {
        const double b = 2.0 * sg * m / ((2.0 * sg - 1.0) * kPi);
        const double t = kPi * k / n;
        return std::sqrt(kPi * b) * std::exp(-b * t * t);
    }
    const double b = kPi * (2.0 - 1.0 / sg);
    const double om = 2.0 * kPi * k / n;
    const double arg2 = b * b - om * om;   // > 0 for |k| <= M/2 = n/(2 sigma), sigma > 1
    return kPi * m / std::sinh(b * m) * bessel_i0_series(m * std::sqrt(arg2 > 0 ? arg2 : 0.0));
}

void fill_window_params(enuf_plan* p) {
    enuf::WindowParams& w = p->wp;
    w.kind = p->window;
    w.m = p->m;
    if (p->window == ENUF_WINDOW_SINC_POWER) {
        w.b = kPi * (2.0 - 1.0 / p->sigma) / (2.0 * p->m);   // phi = sinc(b d)^2m
        w.inv_b = w.bm = w.inv1m = w.A = 0.0;
    } else if (p->window == ENUF_WINDOW_BSPLINE) {
        w.b = w.inv_b = w.bm = w.inv1m = 0.0;
        w.A = 1.0 / bspline_host(2 * p->m, 0.0);       // phi = A B_2m
    } else if (p->window == ENUF_WINDOW_GAUSSIAN) {
        w.b = 2.0 * p->sigma * p->m / ((2.0 * p->sigma - 1.0) * kPi);
        w.inv_b = 1.0 / w.b;
        w.bm = w.b * p->m;
        w.inv1m = 1.0;
        w.A = 0.0;
    } else {
        w.b = kPi * (2.0 - 1.0 / p->sigma);
        w.inv_b = 1.0 / w.b;
        w.bm = w.b * p->m;
        w.inv1m = 1.0 / (1.0 - std::exp(-2.0 * w.bm));
        w.A = p->m / std::sinh(w.bm);
    }
}

// The window and its analytic continuation beyond |d| = m (Kaiser-Bessel:
// sinh(b s)/s with s^2 = m^2 - d^2 < 0 becomes sin(b t)/t, t^2 = d^2 - m^2), phi(0) = 1.
// Only used to fit the polynomial table: the kernels cut the support themselves.
double window_smooth(const enuf_plan* p, double d) {
    const double m = p->m, sg = p->sigma;
    if (p->window == ENUF_WINDOW_SINC_POWER) {
        const double t = kPi * (2.0 - 1.0 / sg) / (2.0 * m) * d;
        return std::pow(t == 0.0 ? 1.0 : std::sin(t) / t, 2 * p->m);
    }
    if (p->window == ENUF_WINDOW_GAUSSIAN) {
        const double b = 2.0 * sg * m / ((2.0 * sg - 1.0) * kPi);
        return std::exp(-d * d / b);
    }
    const double b = kPi * (2.0 - 1.0 / sg), A = m / std::sinh(b * m);
    const double s2 = (m - d) * (m + d), z = b * b * s2;
    if (std::fabs(z) < 1e-2)   // sinh(x)/x = 1 + x^2/6 + x^4/120 + x^6/5040 + x^8/362880, x^2 = z
        return A * b * (1.0 + z * (1.0 / 6.0 + z * (1.0 / 120.0 + z * (1.0 / 5040.0 + z / 362880.0))));
    if (s2 > 0) { const double s = std::sqrt(s2); return A * std::sinh(b * s) / s; }
    const double t = std::sqrt(-s2);
    return A * std::sin(b * t) / t;
}

// Step a0 (fp32 path): for each stencil offset j = 0..m the Chebyshev interpolant of degree
// D = poly_degree(m) of d0 -> phi(d0 - j) on [-1/2, 1/2], converted to monomials in d0, and
// its exact derivative (enuf_common.cuh, PolyArg).
void build_poly_table(enuf_plan* p) {
    if (p->window == ENUF_WINDOW_BSPLINE) {
        // exact pieces: phi(t - j) = sum_i B^(i)(-j from the right) / i! t^i on t in [0, 1/2], degree 2m - 1
        const int P = 2 * p->m;
        const double A = 1.0 / bspline_host(P, 0.0);
        for (int jj = 0; jj <= 2 * p->m; ++jj) {
            const int j = jj - p->m;
            double fact = 1.0, c[16] = {0};
            for (int i = 0; i < P; ++i) {
                if (i > 0) fact *= i;
                c[i] = A * bspline_deriv_host(P, i, (double)-j) / fact;
            }
            for (int i = 0; i < P; ++i) {
                p->bs_c[i][jj] = (float)c[i];
                p->bs_d[i][jj] = i + 1 < P ? (float)((i + 1) * c[i + 1]) : 0.f;
            }
        }
        return;
    }
    constexpr int NCMAX = enuf::kPolyMaxDeg + 1;
    const int D = enuf::poly_degree(p->m), NC = D + 1;
    for (int j = 0; j <= p->m; ++j) {
        long double a[NCMAX];
        for (int k = 0; k < NC; ++k) {
            long double acc = 0;
            for (int i = 0; i < NC; ++i) {
                const double th = kPi * (i + 0.5) / NC;
                acc += (long double)window_smooth(p, 0.5 * std::cos(th) - j) * std::cos(k * th);
            }
            a[k] = acc * (k == 0 ? 1.0L : 2.0L) / NC;
        }
        // T_0 = 1, T_1 = 2t, T_{k+1} = 4t T_k - T_{k-1} (x = 2t)
        long double c[NCMAX] = {0}, t0[NCMAX] = {0}, t1[NCMAX] = {0}, t2[NCMAX];
        t0[0] = 1; t1[1] = 2;
        for (int e = 0; e < NC; ++e) c[e] = a[0] * t0[e] + a[1] * t1[e];
        for (int k = 2; k < NC; ++k) {
            for (int e = 0; e < NC; ++e) t2[e] = (e > 0 ? 4 * t1[e - 1] : 0.0L) - t0[e];
            for (int e = 0; e < NC; ++e) { c[e] += a[k] * t2[e]; t0[e] = t1[e]; t1[e] = t2[e]; }
        }
        for (int k = 0; k < NC; ++k) p->poly_c[k][j] = (float)c[k];
        for (int k = 0; k < D; ++k) p->poly_d[k][j] = (float)((k + 1) * c[k + 1]);
    }
}

template <typename T>
int upload(void* dst, const std::vector<double>& src, cudaStream_t s) {
    std::vector<T> tmp(src.size());
    for (size_t i = 0; i < src.size(); ++i) tmp[i] = (T)src[i];
    CU(cudaMemcpyAsync(dst, tmp.data(), sizeof(T) * tmp.size(), cudaMemcpyHostToDevice, s));
    CU(cudaStreamSynchronize(s));
    return ENUF_OK;
}

// Step a0: twiddles, 1/Phi(k), f^2 w(|n|^2) in fp64 on the host, rounded once to T.
int build_tables(enuf_plan* p) {
    fill_window_params(p);
    const int n = p->n, kc = p->k_cut;
    // twiddles of the four-step FFT, one table per direction, laid out [k1][a] (enuf_fft.cuh):
    // forward (RA, RB) = (16, n/16), inverse (n/16, 16); entry = exp(-2 pi i a k1 / n)
    std::vector<double> tw(4 * (size_t)n), iphi((size_t)kc + 1), wf((size_t)kc * kc + 1);
    if (p->mixed) {
        // plain table exp(-2 pi i j / n), j < n (enuf_fft_mixed.cuh)
        for (int j = 0; j < n; ++j) { tw[2 * j] = std::cos(2.0 * kPi * j / n); tw[2 * j + 1] = -std::sin(2.0 * kPi * j / n); }
    }
    for (int dir = 0; dir < 2 && !p->mixed; ++dir) {
        const int RA = dir == 0 ? 16 : n / 16, RB = n / RA;
        for (int k1 = 0; k1 < RA; ++k1)
            for (int a = 0; a < RB; ++a) {
                const size_t e = (size_t)dir * n + (size_t)k1 * RB + a;
                const int j = (a * k1) % n;
                tw[2 * e] = std::cos(2.0 * kPi * j / n);
                tw[2 * e + 1] = -std::sin(2.0 * kPi * j / n);
            }
    }
    for (int k = 0; k <= kc; ++k) iphi[k] = 1.0 / window_transform(p, k);
    wf[0] = 0.0;
    const double a = kPi / (p->alpha * p->L), tl = kPi * p->lambda / p->L;
    for (int s = 1; s <= kc * kc; ++s) {
        double w = std::exp(-a * a * s) / s;                    // Eq. 38
        if (p->lambda != 0.0) {                                 // R19: (1 + (pi lambda |n|/L)^2)^-4
            const double g = 1.0 + tl * tl * s;
            w /= (g * g) * (g * g);
        }
        wf[s] = w;
    }
    int rc;
    build_poly_table(p);
    if (p->precision == ENUF_F32) {
        if ((rc = upload<float>(p->tw, tw, p->stream))) return rc;
        if ((rc = upload<float>(p->iphi, iphi, p->stream))) return rc;
        if ((rc = upload<float>(p->wf, wf, p->stream))) return rc;
    } else {
        if ((rc = upload<double>(p->tw, tw, p->stream))) return rc;
        if ((rc = upload<double>(p->iphi, iphi, p->stream))) return rc;
        if ((rc = upload<double>(p->wf, wf, p->stream))) return rc;
    }
    p->tables_dirty = false;
    return ENUF_OK;
}

int dev_alloc(enuf_plan* p, void** ptr, size_t bytes) {
    if (bytes == 0) bytes = 16;
    cudaError_t e = cudaMalloc(ptr, bytes);
    if (e != cudaSuccess) {
        *ptr = nullptr;
        (void)cudaGetLastError();
        return e == cudaErrorMemoryAllocation ? fail(ENUF_ENOMEM, "cudaMalloc(%zu) failed: out of device memory", bytes)
                                              : fail_cuda(e, "cudaMalloc");
    }
    p->workspace_bytes += bytes;
    return ENUF_OK;
}

void drop_graph(enuf_plan* p) {
    if (p->gexec) { cudaGraphExecDestroy(p->gexec); p->gexec = nullptr; }
    p->g_r = p->g_q = nullptr; p->g_F = nullptr; p->g_N = -1;
}

void free_workspace(enuf_plan* p) {
    drop_graph(p);
    auto fr = [](void* q) { if (q) cudaFree(q); };
    fr(p->rec); fr(p->rows); p->rows = nullptr; fr(p->binrank); p->binrank = nullptr; fr(p->bin_count); fr(p->bin_offset); fr(p->bin_cursor);
    fr(p->scan_total); fr(p->scan_desc); p->scan_desc = nullptr; fr(p->scan_epoch); p->scan_epoch = nullptr;
    for (int d = 0; d < 3; ++d) { fr(p->grid[d]); fr(p->A1[d]); fr(p->A2[d]); p->grid[d] = p->A1[d] = p->A2[d] = nullptr; }
    fr(p->spectrum); fr(p->tw); fr(p->iphi); fr(p->wf); fr(p->e_partial); fr(p->e_dev); fr(p->fft_done);
    fr(p->r_stage); fr(p->q_stage); fr(p->F_stage);
    fr(p->real_pos); fr(p->real_idx); fr(p->real_count); fr(p->real_offset); fr(p->real_cursor);
    fr(p->real_scan_total); fr(p->real_partial); fr(p->real_e_dev);
    if (p->real_e_pinned) cudaFreeHost(p->real_e_pinned);
    p->real_pos = nullptr; p->real_idx = p->real_count = p->real_offset = p->real_cursor = p->real_scan_total = nullptr;
    p->real_partial = p->real_e_dev = p->real_e_pinned = nullptr;
    p->real_ncells_cap = 0;
    if (p->e_pinned) cudaFreeHost(p->e_pinned);
    if (p->ev_ring) {
        for (int i = 0; i < enuf_plan::kProfRing * enuf_plan::kProfEv; ++i)
            if (p->ev_ring[i]) cudaEventDestroy(p->ev_ring[i]);
        delete[] p->ev_ring;
        p->ev_ring = p->ev = nullptr;
    }
    p->prof_evals = 0;
    p->rec = p->spectrum = p->tw = p->iphi = p->wf = p->r_stage = p->q_stage = p->F_stage = nullptr;
    p->bin_count = p->bin_offset = p->bin_cursor = p->scan_total = nullptr;
    p->e_partial = p->e_dev = p->e_pinned = nullptr;
    p->fft_done = nullptr;
    p->events_valid = false;
    p->partial_ready = false;
    p->evaluated = false;          // e_dev, grid, spectrum are gone
    p->q_stage_valid = false;
    p->bin_count_clean = false;
    p->real_count_clean = false;
    p->allocated = false;
    p->workspace_bytes = 0;
    (void)cudaGetLastError();
}

// Allocate everything that depends on precision / variant (lazily, at the first evaluation).
int ensure_allocated(enuf_plan* p) {
    if (p->allocated) return ENUF_OK;
    int dev_count = 0;
    cudaError_t e = cudaGetDeviceCount(&dev_count);
    if (e != cudaSuccess || dev_count == 0) {
        (void)cudaGetLastError();
        return fail(ENUF_ECUDA, "no CUDA device available (%s); this library has no CPU fallback",
                    e != cudaSuccess ? cudaGetErrorString(e) : "device count 0");
    }
    p->esize = p->precision == ENUF_F32 ? 4 : 8;
    {
        int dev = 0, sms = 0;
        if (cudaGetDevice(&dev) == cudaSuccess &&
            cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev) == cudaSuccess && sms > 0)
            p->num_sms = sms;
        (void)cudaGetLastError();
    }
    // the outermost stencil point on the far side of a particle is an exact zero for Kaiser-Bessel;
    // only when the particle sits exactly on a grid point are both ends non-zero, with the value
    // b m / sinh(b m) (<= 2.7e-9 for m >= 5): the fp32 kernels then skip that point
    p->trim = p->precision == ENUF_F32 && p->window == ENUF_WINDOW_KAISER_BESSEL && p->m >= 5;
    p->tg.trim = p->trim ? 1 : 0;
    const size_t es = p->esize, n = p->n, n3 = n * n * n, cap = (size_t)(p->N_cap > 0 ? p->N_cap : 1);
    const int nfield = p->variant == ENUF_FORCE_IK ? 3 : 1;
    int rc;
#define ALLOC(ptr, bytes) if ((rc = dev_alloc(p, (void**)&(ptr), (bytes)))) { free_workspace(p); return rc; }
    ALLOC(p->rec, (es == 4 ? sizeof(enuf::PSlot<float>) : sizeof(enuf::PSlot<double>)) * cap);
    ALLOC(p->rows, es * 48 * cap);
    ALLOC(p->bin_count, 4 * (size_t)p->tg.nbins);
    ALLOC(p->bin_offset, 4 * ((size_t)p->tg.nbins + 1));
    ALLOC(p->bin_cursor, 4 * (size_t)p->tg.nbins);
    ALLOC(p->binrank, 8 * cap);
    ALLOC(p->scan_total, 4 * (((size_t)p->tg.nbins + 1023) / 1024));
    ALLOC(p->scan_desc, 8 * (((size_t)p->tg.nbins + 1023) / 1024));
    ALLOC(p->scan_epoch, 4);
    for (int d = 0; d < nfield; ++d) {
        ALLOC(p->grid[d], es * n3);
        // (mixed-radix grids: A1 is the full complex n^3 spectrum, A2 is not used)
        ALLOC(p->A1[d], p->mixed ? 2 * es * n3 : 2 * es * n * n * p->Kxp);
        ALLOC(p->A2[d], p->mixed ? 16 : 2 * es * n * p->Ky * p->Kxp);
    }
    if (p->keep_spectrum) ALLOC(p->spectrum, 2 * es * (size_t)p->Ky * p->Ky * p->Kxp);
    ALLOC(p->tw, 4 * es * n);
    ALLOC(p->iphi, es * ((size_t)p->k_cut + 1));
    ALLOC(p->wf, es * ((size_t)p->k_cut * p->k_cut + 1));
    const int lpc = 256 / (p->n / 16 > 0 ? p->n / 16 : 1);
    p->n_partial = p->mixed ? enuf_plan::kMixedScaleCtas : (int)(((size_t)p->Ky * p->Kxp + lpc - 1) / lpc);
    ALLOC(p->e_partial, 8 * (size_t)p->n_partial);
    ALLOC(p->e_dev, 8);
    ALLOC(p->fft_done, 4);
#undef ALLOC
    if (cudaMallocHost((void**)&p->e_pinned, 8) != cudaSuccess) {
        (void)cudaGetLastError();
        free_workspace(p);
        return fail(ENUF_ENOMEM, "cudaMallocHost failed");
    }
    p->ev_ring = new (std::nothrow) cudaEvent_t[enuf_plan::kProfRing * enuf_plan::kProfEv]();
    if (!p->ev_ring) { free_workspace(p); return fail(ENUF_ENOMEM, "out of host memory"); }
    for (int i = 0; i < enuf_plan::kProfRing * enuf_plan::kProfEv; ++i) {
        if (cudaEventCreate(&p->ev_ring[i]) != cudaSuccess) { free_workspace(p); return fail(ENUF_ECUDA, "cudaEventCreate failed"); }
    }
    p->ev = p->ev_ring;
    p->prof_evals = 0;
    p->events_valid = true;
    // pad columns of A1/A2 (kx in (k_cut, Kxp)) must hold finite values
    for (int d = 0; d < nfield; ++d) {
        cudaMemsetAsync(p->A1[d], 0, p->mixed ? 2 * es * n3 : 2 * es * n * n * p->Kxp, p->stream);
        cudaMemsetAsync(p->A2[d], 0, p->mixed ? 16 : 2 * es * n * p->Ky * p->Kxp, p->stream);
    }
    if (p->spectrum) cudaMemsetAsync(p->spectrum, 0, 2 * es * (size_t)p->Ky * p->Ky * p->Kxp, p->stream);
    cudaMemsetAsync(p->e_dev, 0, 8, p->stream);
    cudaMemsetAsync(p->fft_done, 0, 4, p->stream);
    cudaMemsetAsync(p->scan_desc, 0, 8 * (((size_t)p->tg.nbins + 1023) / 1024), p->stream);
    cudaMemsetAsync(p->scan_epoch, 0, 4, p->stream);
    rc = p->precision == ENUF_F32 ? enuf::configure_kernels<float>(p) : enuf::configure_kernels<double>(p);
    if (rc) {
        cudaError_t le = cudaGetLastError();
        free_workspace(p);
        return fail_cuda(le, "cudaFuncSetAttribute(max dynamic shared memory)");
    }
    p->allocated = true;
    p->tables_dirty = true;
    return ENUF_OK;
}

int prepare(enuf_plan* p) {
    int rc = ensure_allocated(p);
    if (rc) return rc;
    if (p->tables_dirty && (rc = build_tables(p))) return rc;
    return ENUF_OK;
}

template <typename T>
int run_bin_spread(enuf_plan* p, const void* r, const void* q, void* F) {
    int l = enuf::launch_bin<T>(p, r, q, F);
    if (l < 0) return -1;
    p->launches += l;
    if (p->profile) cudaEventRecord(p->ev[1], p->stream);
    {
        // mean number of particles a spreading CTA stages per slab: N (column + stencil margin) / n^3
        const int w = 2 * p->m - (p->trim ? 1 : 0), cx = 8 * p->spread_npx + w, cy = 16 + w;
        const double per_slab = (double)p->N * cx * cy / ((double)p->n * p->n * p->n);
        p->spread_sparse = sizeof(T) == 4 && (p->spread_sparse_user < 0 ? per_slab <= 12.0 : p->spread_sparse_user == 1);
    }
    l = enuf::launch_spread<T>(p);
    if (l < 0) return -1;
    p->launches += l;
    if (p->profile) cudaEventRecord(p->ev[2], p->stream);
    return 0;
}

template <typename T>
int run_all(enuf_plan* p, const void* r, const void* q, void* F) {
    if (p->profile) cudaEventRecord(p->ev[0], p->stream);
    if (run_bin_spread<T>(p, r, q, F)) return -1;
    int l = enuf::launch_fft<T>(p);
    if (l < 0) return -1;
    p->launches += l;
    if (p->profile) cudaEventRecord(p->ev[3], p->stream);
    l = enuf::launch_gather<T>(p, F);
    if (l < 0) return -1;
    p->launches += l;
    if (p->profile) { cudaEventRecord(p->ev[4], p->stream); cudaEventRecord(p->ev[5], p->stream); }
    return 0;
}

// Multi-GPU halves (enuf.h, "Sharded evaluation"): a1 + a2 + the X, Y forward passes ...
template <typename T>
int run_partial(enuf_plan* p, const void* r, const void* q, void* F) {
    if (p->profile) cudaEventRecord(p->ev[0], p->stream);
    if (run_bin_spread<T>(p, r, q, F)) return -1;
    const int l = enuf::launch_fft_forward<T>(p);
    if (l < 0) return -1;
    p->launches += l;
    return 0;
}

// ... and Z forward . scale . energy . Z inverse, Y and X inverse passes, gather (a4 .. a7)
template <typename T>
int run_finish(enuf_plan* p, void* F) {
    int l = enuf::launch_fft_backward<T>(p);
    if (l < 0) return -1;
    p->launches += l;
    if (p->profile) cudaEventRecord(p->ev[3], p->stream);
    l = enuf::launch_gather<T>(p, F);
    if (l < 0) return -1;
    p->launches += l;
    if (p->profile) { cudaEventRecord(p->ev[4], p->stream); cudaEventRecord(p->ev[5], p->stream); }
    return 0;
}

int evaluate_device(enuf_plan* p, const void* r, const void* q, void* F, double* E) {
    p->launches = 0;
    if (p->profile) {
        p->ev = p->ev_ring + (p->prof_evals % enuf_plan::kProfRing) * enuf_plan::kProfEv;
        ++p->prof_evals;
    }
    if (p->N == 0) {
        CU(cudaMemsetAsync(p->e_dev, 0, 8, p->stream));
        if (p->profile) for (int i = 0; i <= ENUF_NUM_STAGES; ++i) cudaEventRecord(p->ev[i], p->stream);
    } else if (p->use_graph && !p->profile && p->gexec && r == p->g_r && q == p->g_q && F == p->g_F && p->N == p->g_N) {
        CU(cudaGraphLaunch(p->gexec, p->stream));
        p->launches = p->g_launches;
    } else if (p->use_graph && !p->profile && p->evaluated && r == p->g_r && q == p->g_q && F == p->g_F && p->N == p->g_N) {
        // second call with the same arguments: capture (nothing runs), instantiate, launch.  The capture is
        // made on a stream of the plan's own, because the caller's may be the legacy default stream.
        if (!p->cap_stream) CU(cudaStreamCreateWithFlags(&p->cap_stream, cudaStreamNonBlocking));
        cudaStream_t user = p->stream;
        p->stream = p->cap_stream;
        cudaGraph_t graph = nullptr;
        cudaError_t ce = cudaStreamBeginCapture(p->cap_stream, cudaStreamCaptureModeThreadLocal);
        int rc = 0;
        if (ce == cudaSuccess) {
            rc = p->precision == ENUF_F32 ? run_all<float>(p, r, q, F) : run_all<double>(p, r, q, F);
            ce = cudaStreamEndCapture(p->cap_stream, &graph);
        }
        p->stream = user;
        if (ce != cudaSuccess || rc || !graph) {
            if (graph) cudaGraphDestroy(graph);
            drop_graph(p);
            return fail_cuda(ce != cudaSuccess ? ce : (p->launch_error != cudaSuccess ? p->launch_error : cudaErrorUnknown),
                             "CUDA graph capture");
        }
        ce = cudaGraphInstantiate(&p->gexec, graph, 0);
        cudaGraphDestroy(graph);
        if (ce != cudaSuccess) { p->gexec = nullptr; drop_graph(p); return fail_cuda(ce, "cudaGraphInstantiate"); }
        p->g_launches = p->launches;
        CU(cudaGraphLaunch(p->gexec, p->stream));
    } else {
        if (p->use_graph) { drop_graph(p); p->g_r = r; p->g_q = q; p->g_F = F; p->g_N = p->N; }
        int rc = p->precision == ENUF_F32 ? run_all<float>(p, r, q, F) : run_all<double>(p, r, q, F);
        if (rc) return fail_launch(p);
    }
    p->evaluated = true;
    if (E) {
        CU(cudaMemcpyAsync(p->e_pinned, p->e_dev, 8, cudaMemcpyDeviceToHost, p->stream));
        CU(cudaStreamSynchronize(p->stream));
        *E = *p->e_pinned;
    }
    return ENUF_OK;
}

}  // namespace

extern "C" {

const char* enuf_last_error(void) { return g_err; }

int enuf_plan_create(enuf_plan** out, int64_t N, double L, double alpha, int k_cut, int M, double sigma, int m) {
    const double Lb[3] = {L, L, L};
    return enuf_plan_create_box(out, N, Lb, alpha, k_cut, M, sigma, m);
}

int enuf_plan_create_box(enuf_plan** out, int64_t N, const double* Lb, double alpha, int k_cut, int M, double sigma,
                         int m) {
    g_err[0] = 0;
    if (!out) return fail(ENUF_EINVAL, "out is NULL");
    *out = nullptr;
    if (!Lb) return fail(ENUF_EINVAL, "Lb is NULL");
    if (N < 0 || N > 0xFFFFFFFFll) return fail(ENUF_EINVAL, "N = %lld out of range [0, 2^32)", (long long)N);
    for (int d = 0; d < 3; ++d)
        if (!(Lb[d] > 0) || !std::isfinite(Lb[d])) return fail(ENUF_EINVAL, "L must be positive and finite");
    const double L = Lb[0];
    if (!(alpha > 0) || !std::isfinite(alpha)) return fail(ENUF_EINVAL, "alpha must be positive and finite");
    if (M < 2) return fail(ENUF_EINVAL, "M must be >= 2");
    if (!(sigma > 1.0) || !std::isfinite(sigma)) return fail(ENUF_EINVAL, "sigma must be > 1");
    const double nd = sigma * M;
    const int n = (int)std::lround(nd);
    const bool pow2 = n == 32 || n == 64 || n == 128 || n == 256, mixed = n == 48 || n == 96 || n == 192 || n == 384;
    if (std::fabs(nd - n) > 1e-9 || !(pow2 || mixed))
        return fail(ENUF_EINVAL, "sigma*M = %g must be one of 32, 64, 128, 256 or 48, 96, 192, 384", nd);
    if (k_cut < 1 || 2 * k_cut > M) return fail(ENUF_EINVAL, "k_cut = %d must satisfy 1 <= k_cut <= M/2 = %d", k_cut, M / 2);
    if (m < 1 || m > enuf::kMaxM) return fail(ENUF_EINVAL, "m = %d must satisfy 1 <= m <= %d", m, enuf::kMaxM);
    enuf_plan* p = new (std::nothrow) enuf_plan();
    if (!p) return fail(ENUF_ENOMEM, "out of host memory");
    p->N_cap = p->N = N;
    p->L = L; p->alpha = alpha; p->sigma = sigma; p->k_cut = k_cut; p->M = M; p->n = n; p->m = m;
    p->mixed = mixed;
    for (int d = 0; d < 3; ++d) p->Lb[d] = Lb[d];
    p->box = !(Lb[0] == Lb[1] && Lb[1] == Lb[2]);
    p->tg.n = n;
    p->tg.nt = n / enuf::kTile;
    p->tg.nbins = p->tg.nt * p->tg.nt * n;
    p->spread_npx = n >= 128 ? 4 : 2;
    p->zchunk = n;                 // only used when set through ENUF_OPT_SPREAD_ZCHUNK
    p->Kxp = ((k_cut + 1 + enuf::kLinesPerGroup - 1) / enuf::kLinesPerGroup) * enuf::kLinesPerGroup;
    p->Ky = 2 * k_cut + 1;
    fill_window_params(p);
    *out = p;
    return ENUF_OK;
}

int enuf_plan_set(enuf_plan* p, int key, double value) {
    g_err[0] = 0;
    if (!p) return fail(ENUF_EINVAL, "plan is NULL");
    drop_graph(p);                 // whatever changes, a captured evaluation no longer describes the plan
    p->partial_ready = false;      // ... nor does a partial spectrum: enuf_forces_from_spectrum needs a fresh first half
    const int iv = (int)value;
    switch (key) {
        case ENUF_OPT_PRECISION:
            if (iv != ENUF_F32 && iv != ENUF_F64) return fail(ENUF_EINVAL, "precision must be ENUF_F32 or ENUF_F64");
            if (p->allocated && iv != p->precision) return fail(ENUF_ESTATE, "precision is fixed after the first evaluation");
            p->precision = iv;
            return ENUF_OK;
        case ENUF_OPT_WINDOW:
            if (iv != ENUF_WINDOW_GAUSSIAN && iv != ENUF_WINDOW_KAISER_BESSEL && iv != ENUF_WINDOW_BSPLINE &&
                iv != ENUF_WINDOW_SINC_POWER)
                return fail(ENUF_EINVAL, "unknown window");
            p->window = iv; p->tables_dirty = true; fill_window_params(p);
            p->trim = p->precision == ENUF_F32 && p->window == ENUF_WINDOW_KAISER_BESSEL && p->m >= 5;
            p->tg.trim = p->trim ? 1 : 0;
            return ENUF_OK;
        case ENUF_OPT_FORCE_VARIANT:
            if (iv != ENUF_FORCE_ANALYTIC && iv != ENUF_FORCE_IK) return fail(ENUF_EINVAL, "unknown force variant");
            if (p->allocated && iv != p->variant) { cudaStreamSynchronize(p->stream); free_workspace(p); }
            p->variant = iv;
            return ENUF_OK;
        case ENUF_OPT_SLATER_LAMBDA:
            if (!(value >= 0) || !std::isfinite(value)) return fail(ENUF_EINVAL, "lambda must be >= 0");
            p->lambda = value; p->tables_dirty = true;
            return ENUF_OK;
        case ENUF_OPT_NUM_PARTICLES:
            if (value < 0 || value > (double)p->N_cap || value != std::floor(value))
                return fail(ENUF_EINVAL, "N must be an integer in [0, %lld]", (long long)p->N_cap);
            p->N = (int64_t)value;
            return ENUF_OK;
        case ENUF_OPT_PROFILE:
            p->profile = iv != 0;
            p->prof_evals = 0;
            return ENUF_OK;
        case ENUF_OPT_KEEP_SPECTRUM:
            if (p->allocated && (iv != 0) != p->keep_spectrum) { cudaStreamSynchronize(p->stream); free_workspace(p); }
            p->keep_spectrum = iv != 0;
            return ENUF_OK;
        case ENUF_OPT_CUDA_GRAPH:
            p->use_graph = iv != 0;
            return ENUF_OK;
        case ENUF_OPT_PDL:
            p->pdl = iv != 0;
            return ENUF_OK;
        case ENUF_OPT_SPREAD_SPARSE:
            if (iv < -1 || iv > 1) return fail(ENUF_EINVAL, "spread_sparse must be -1 (auto), 0 or 1");
            p->spread_sparse_user = iv;
            return ENUF_OK;
        case ENUF_OPT_SPREAD_ZCHUNK:
            if (iv < 1 || iv > p->n) return fail(ENUF_EINVAL, "zchunk must be an integer in [1, n]");
            p->zchunk = iv; p->zchunk_user = true;
            return ENUF_OK;
        default:
            return fail(ENUF_EINVAL, "unknown option key %d", key);
    }
}

int enuf_plan_set_stream(enuf_plan* p, void* cuda_stream) {
    g_err[0] = 0;
    if (!p) return fail(ENUF_EINVAL, "plan is NULL");
    p->stream = static_cast<cudaStream_t>(cuda_stream);
    return ENUF_OK;
}

int enuf_energy_forces(enuf_plan* p, const void* r, const void* q, void* F, double* E) {
    g_err[0] = 0;
    if (!p) return fail(ENUF_EINVAL, "plan is NULL");
    if (p->N > 0 && (!r || !q || !F)) return fail(ENUF_EINVAL, "r, q and F must be non-NULL when N > 0");
    int rc = prepare(p);
    if (rc) return rc;
    return evaluate_device(p, r, q, F, E);
}

int enuf_energy_forces_host(enuf_plan* p, const void* r_host, const void* q_host, void* F_host, double* E) {
    g_err[0] = 0;
    if (!p) return fail(ENUF_EINVAL, "plan is NULL");
    if (p->N > 0 && (!r_host || !F_host)) return fail(ENUF_EINVAL, "r and F must be non-NULL when N > 0");
    int rc = prepare(p);
    if (rc) return rc;
    if (p->N > 0 && !q_host && !p->q_stage_valid)
        return fail(ENUF_ESTATE, "q_host = NULL reuses the charges of the previous host call: there is none");
    const size_t es = p->esize, cap = (size_t)(p->N_cap > 0 ? p->N_cap : 1);
    if (!p->r_stage) {
        // the three staging buffers are allocated as a group: all or none
        if ((rc = dev_alloc(p, &p->r_stage, 3 * es * cap)) || (rc = dev_alloc(p, &p->q_stage, es * cap)) ||
            (rc = dev_alloc(p, &p->F_stage, 3 * es * cap))) {
            if (p->r_stage) cudaFree(p->r_stage);
            if (p->q_stage) cudaFree(p->q_stage);
            if (p->F_stage) cudaFree(p->F_stage);
            p->r_stage = p->q_stage = p->F_stage = nullptr;
            return rc;
        }
    }
    const size_t N = (size_t)p->N;
    if (N > 0) {
        CU(cudaMemcpyAsync(p->r_stage, r_host, 3 * es * N, cudaMemcpyHostToDevice, p->stream));
        if (q_host) {
            CU(cudaMemcpyAsync(p->q_stage, q_host, es * N, cudaMemcpyHostToDevice, p->stream));
            p->q_stage_valid = true;
        }
    }
    rc = evaluate_device(p, p->r_stage, p->q_stage, p->F_stage, nullptr);
    if (rc) return rc;
    if (N > 0) CU(cudaMemcpyAsync(F_host, p->F_stage, 3 * es * N, cudaMemcpyDeviceToHost, p->stream));
    CU(cudaMemcpyAsync(p->e_pinned, p->e_dev, 8, cudaMemcpyDeviceToHost, p->stream));
    CU(cudaStreamSynchronize(p->stream));
    if (E) *E = *p->e_pinned;
    return ENUF_OK;
}

int enuf_spectrum_partial(enuf_plan* p, const void* r, const void* q, void* F) {
    g_err[0] = 0;
    if (!p) return fail(ENUF_EINVAL, "plan is NULL");
    if (p->N > 0 && (!r || !q || !F)) return fail(ENUF_EINVAL, "r, q and F must be non-NULL when N > 0");
    int rc = prepare(p);
    if (rc) return rc;
    p->launches = 0;
    p->partial_ready = false;
    if (p->profile) {
        p->ev = p->ev_ring + (p->prof_evals % enuf_plan::kProfRing) * enuf_plan::kProfEv;
        ++p->prof_evals;
    }
    if (p->N == 0) {
        // no particles on this rank: its partial spectrum is zero
        if (p->mixed) CU(cudaMemsetAsync(p->A1[0], 0, 2 * p->esize * (size_t)p->n * p->n * p->n, p->stream));
        else CU(cudaMemsetAsync(p->A2[0], 0, 2 * p->esize * (size_t)p->n * p->Ky * p->Kxp, p->stream));
        if (p->profile) for (int i = 0; i <= 2; ++i) cudaEventRecord(p->ev[i], p->stream);
    } else {
        rc = p->precision == ENUF_F32 ? run_partial<float>(p, r, q, F) : run_partial<double>(p, r, q, F);
        if (rc) return fail_launch(p);
    }
    p->partial_ready = true;
    return ENUF_OK;
}

int enuf_plan_spectrum_buffer(enuf_plan* p, void** dev_ptr, size_t* count) {
    g_err[0] = 0;
    if (!p || !dev_ptr || !count) return fail(ENUF_EINVAL, "plan, dev_ptr or count is NULL");
    int rc = prepare(p);
    if (rc) return rc;
    // (grids of 3 * 2^k points: the full complex n^3 spectrum after the three forward passes)
    *dev_ptr = p->mixed ? p->A1[0] : p->A2[0];
    *count = p->mixed ? 2 * (size_t)p->n * p->n * p->n : 2 * (size_t)p->n * p->Ky * p->Kxp;
    return ENUF_OK;
}

int enuf_forces_from_spectrum(enuf_plan* p, void* F, double* E) {
    g_err[0] = 0;
    if (!p) return fail(ENUF_EINVAL, "plan is NULL");
    if (!p->allocated || p->tables_dirty || !p->partial_ready)
        return fail(ENUF_ESTATE, "enuf_forces_from_spectrum needs a preceding enuf_spectrum_partial (and no enuf_plan_set since)");
    if (p->N > 0 && !F) return fail(ENUF_EINVAL, "F must be non-NULL when N > 0");
    p->partial_ready = false;
    const int before = p->launches;
    int rc;
    if (p->N == 0) {
        // no particles to interpolate onto, but the energy of the summed spectrum is still produced
        rc = p->precision == ENUF_F32 ? enuf::launch_fft_backward<float>(p) : enuf::launch_fft_backward<double>(p);
        if (rc < 0) return fail_launch(p);
        p->launches = before + rc;
        if (p->profile) for (int i = 3; i <= ENUF_NUM_STAGES; ++i) cudaEventRecord(p->ev[i], p->stream);
    } else {
        rc = p->precision == ENUF_F32 ? run_finish<float>(p, F) : run_finish<double>(p, F);
        if (rc) return fail_launch(p);
    }
    p->evaluated = true;
    if (E) {
        CU(cudaMemcpyAsync(p->e_pinned, p->e_dev, 8, cudaMemcpyDeviceToHost, p->stream));
        CU(cudaStreamSynchronize(p->stream));
        *E = *p->e_pinned;
    }
    return ENUF_OK;
}

namespace {
// Chebyshev interpolant of degree kErfcDeg of g(t) = exp(x^2) erfc(x) / t, x = 2 (1/t - 1), on t in
// [1/(1 + xmax/2), 1], converted to monomials in u = ua t + ub in [-1, 1] (enuf_real.cuh, ErfcFit).
void build_erfc_fit(enuf_plan* p, double xmax) {
    constexpr int D = enuf::kErfcDeg, NC = D + 1;
    const double tmin = 1.0 / (1.0 + 0.5 * xmax), ua = 2.0 / (1.0 - tmin), ub = -(1.0 + tmin) / (1.0 - tmin);
    long double a[NC];
    for (int k = 0; k < NC; ++k) {
        long double acc = 0;
        for (int i = 0; i < NC; ++i) {
            const double th = kPi * (i + 0.5) / NC, u = std::cos(th);
            const double t = (u - ub) / ua, x = 2.0 * (1.0 / t - 1.0);
            acc += (long double)(std::exp(x * x) * std::erfc(x) / t) * std::cos(k * th);
        }
        a[k] = acc * (k == 0 ? 1.0L : 2.0L) / NC;
    }
    // T_0 = 1, T_1 = u, T_{k+1} = 2 u T_k - T_{k-1}
    long double c[NC] = {0}, t0[NC] = {0}, t1[NC] = {0}, t2[NC];
    t0[0] = 1; t1[1] = 1;
    for (int e = 0; e < NC; ++e) c[e] = a[0] * t0[e] + a[1] * t1[e];
    for (int k = 2; k < NC; ++k) {
        for (int e = 0; e < NC; ++e) t2[e] = (e > 0 ? 2 * t1[e - 1] : 0.0L) - t0[e];
        for (int e = 0; e < NC; ++e) { c[e] += a[k] * t2[e]; t0[e] = t1[e]; t1[e] = t2[e]; }
    }
    for (int k = 0; k < NC; ++k) p->erfc_c[k] = (float)c[k];
    p->erfc_ua = (float)ua; p->erfc_ub = (float)ub;
    p->erfc_xmax = xmax;
}
}  // namespace

int enuf_real_space(enuf_plan* p, const void* r, const void* q, double r_cut, int accumulate, void* F,
                    double* E_real, double* E_self) {
    g_err[0] = 0;
    if (!p) return fail(ENUF_EINVAL, "plan is NULL");
    if (p->N > 0 && (!r || !q || !F)) return fail(ENUF_EINVAL, "r, q and F must be non-NULL when N > 0");
    if (p->box) return fail(ENUF_EINVAL, "the real-space part is built for cubic boxes only (DESIGN.md section 11)");
    if (!(r_cut > 0) || !(r_cut <= 0.5 * p->L))
        return fail(ENUF_EINVAL, "r_cut = %g must satisfy 0 < r_cut <= L/2 = %g (minimum image)", r_cut, 0.5 * p->L);
    int rc = prepare(p);
    if (rc) return rc;
    // cells of side L/ncd >= r_cut/2, neighbour range s = 2 cells, needs 2 s + 1 <= ncd; smaller boxes
    // (r_cut > 0.4 L) use one cell, i.e. all minimum-image pairs.  The table is capped at 256^3 cells
    // (cells then are larger than needed, which is still correct).
    int s = 2, ncd = (int)std::floor(2.0 * p->L / r_cut);
    if (ncd < 5) { s = 0; ncd = 1; }
    if (ncd > 256) ncd = 256;
    const int ncells = ncd * ncd * ncd;
    const size_t cap = (size_t)(p->N_cap > 0 ? p->N_cap : 1), es = p->esize;
    if (!p->real_pos) {
        // allocated as a group: all or none
        rc = dev_alloc(p, &p->real_pos, 4 * es * cap);
        if (!rc) rc = dev_alloc(p, (void**)&p->real_idx, 4 * cap);
        if (!rc) rc = dev_alloc(p, (void**)&p->real_partial, 16 * ((cap + 127) / 128));
        if (!rc) rc = dev_alloc(p, (void**)&p->real_e_dev, 16);
        if (!rc && cudaMallocHost((void**)&p->real_e_pinned, 16) != cudaSuccess) {
            (void)cudaGetLastError();
            p->real_e_pinned = nullptr;
            rc = fail(ENUF_ENOMEM, "cudaMallocHost failed");
        }
        if (rc) {
            if (p->real_pos) cudaFree(p->real_pos);
            if (p->real_idx) cudaFree(p->real_idx);
            if (p->real_partial) cudaFree(p->real_partial);
            if (p->real_e_dev) cudaFree(p->real_e_dev);
            p->real_pos = nullptr; p->real_idx = nullptr; p->real_partial = nullptr; p->real_e_dev = nullptr;
            return rc;
        }
    }
    if (ncells > p->real_ncells_cap) {
        CU(cudaStreamSynchronize(p->stream));
        auto drop_cells = [&]() {
            if (p->real_count) cudaFree(p->real_count);
            if (p->real_offset) cudaFree(p->real_offset);
            if (p->real_cursor) cudaFree(p->real_cursor);
            if (p->real_scan_total) cudaFree(p->real_scan_total);
            p->real_count = p->real_offset = p->real_cursor = p->real_scan_total = nullptr;
            p->real_ncells_cap = 0;
        };
        drop_cells();
        rc = dev_alloc(p, (void**)&p->real_count, 4 * (size_t)ncells);
        if (!rc) rc = dev_alloc(p, (void**)&p->real_offset, 4 * ((size_t)ncells + 1));
        if (!rc) rc = dev_alloc(p, (void**)&p->real_cursor, 4 * (size_t)ncells);
        if (!rc) rc = dev_alloc(p, (void**)&p->real_scan_total, 4 * (((size_t)ncells + 1023) / 1024));
        if (rc) { drop_cells(); return rc; }
        p->real_ncells_cap = ncells;
        p->real_count_clean = false;
    }
    p->real_ncd = ncd; p->real_s = s;
    {
        const double xmax = p->alpha * r_cut * 1.0001;       // x = alpha d <= alpha r_cut
        if (xmax > p->erfc_xmax || xmax < 0.5 * p->erfc_xmax) build_erfc_fit(p, xmax);
    }
    p->launches = 0;
    if (p->N == 0) {
        CU(cudaMemsetAsync(p->real_e_dev, 0, 16, p->stream));
    } else {
        const int l = p->precision == ENUF_F32 ? enuf::launch_real<float>(p, r, q, r_cut, accumulate, F)
                                               : enuf::launch_real<double>(p, r, q, r_cut, accumulate, F);
        if (l < 0) return fail_launch(p);
        p->launches = l;
    }
    if (E_real || E_self) {
        CU(cudaMemcpyAsync(p->real_e_pinned, p->real_e_dev, 16, cudaMemcpyDeviceToHost, p->stream));
        CU(cudaStreamSynchronize(p->stream));
        if (E_real) *E_real = p->real_e_pinned[0];
        if (E_self) *E_self = p->real_e_pinned[1];
    }
    return ENUF_OK;
}

int enuf_plan_energy(enuf_plan* p, double* E) {
    g_err[0] = 0;
    if (!p || !E) return fail(ENUF_EINVAL, "plan or E is NULL");
    if (!p->evaluated || !p->allocated || !p->e_dev) return fail(ENUF_ESTATE, "no evaluation has been run");
    CU(cudaMemcpyAsync(p->e_pinned, p->e_dev, 8, cudaMemcpyDeviceToHost, p->stream));
    CU(cudaStreamSynchronize(p->stream));
    *E = *p->e_pinned;
    return ENUF_OK;
}

int enuf_plan_stage_ms(enuf_plan* p, float* ms, int count) {
    g_err[0] = 0;
    if (!p || !ms) return fail(ENUF_EINVAL, "plan or ms is NULL");
    if (!p->profile || !p->evaluated) return fail(ENUF_ESTATE, "needs ENUF_OPT_PROFILE = 1 and one evaluation");
    CU(cudaStreamSynchronize(p->stream));
    // events: 0 start, 1 after bin, 2 after spread, 3 after fft(+energy), 4 after gather, 5 end
    for (int i = 0; i < count && i < ENUF_NUM_STAGES; ++i) {
        float t = 0.f;
        CU(cudaEventElapsedTime(&t, p->ev[i], p->ev[i + 1]));
        ms[i] = t;
    }
    return ENUF_OK;
}

int enuf_plan_stage_ms_mean(enuf_plan* p, float* ms, int count, int* n_evals) {
    g_err[0] = 0;
    if (!p || !ms) return fail(ENUF_EINVAL, "plan or ms is NULL");
    if (!p->profile || p->prof_evals == 0 || !p->ev_ring)
        return fail(ENUF_ESTATE, "needs ENUF_OPT_PROFILE = 1 and one evaluation");
    CU(cudaStreamSynchronize(p->stream));
    const int ne = (int)(p->prof_evals < enuf_plan::kProfRing ? p->prof_evals : enuf_plan::kProfRing);
    double acc[ENUF_NUM_STAGES] = {0, 0, 0, 0, 0};
    for (int e = 0; e < ne; ++e) {
        const cudaEvent_t* ev = p->ev_ring + (size_t)e * enuf_plan::kProfEv;
        for (int i = 0; i < ENUF_NUM_STAGES; ++i) {
            float t = 0.f;
            CU(cudaEventElapsedTime(&t, ev[i], ev[i + 1]));
            acc[i] += t;
        }
    }
    for (int i = 0; i < count && i < ENUF_NUM_STAGES; ++i) ms[i] = (float)(acc[i] / ne);
    if (n_evals) *n_evals = ne;
    return ENUF_OK;
}

int enuf_plan_launch_count(const enuf_plan* p) { return p ? p->launches : 0; }

size_t enuf_plan_workspace_bytes(const enuf_plan* p) { return p ? p->workspace_bytes : 0; }

int enuf_plan_copy_field(enuf_plan* p, void* host_out) {
    g_err[0] = 0;
    if (!p || !host_out) return fail(ENUF_EINVAL, "plan or host_out is NULL");
    if (!p->evaluated || !p->allocated) return fail(ENUF_ESTATE, "no evaluation has been run");
    const size_t n = p->n;
    CU(cudaMemcpyAsync(host_out, p->grid[0], p->esize * n * n * n, cudaMemcpyDeviceToHost, p->stream));
    CU(cudaStreamSynchronize(p->stream));
    return ENUF_OK;
}

int enuf_plan_structure_factor(enuf_plan* p, int64_t count, const int* modes, double* out) {
    g_err[0] = 0;
    if (!p || !modes || !out || count < 0) return fail(ENUF_EINVAL, "bad argument");
    if (!p->keep_spectrum || !p->evaluated || !p->allocated || !p->spectrum)
        return fail(ENUF_ESTATE, "needs ENUF_OPT_KEEP_SPECTRUM = 1 before the evaluation");
    const size_t cnt = (size_t)p->Ky * p->Ky * p->Kxp, es = p->esize;
    std::vector<unsigned char> host(2 * es * cnt);
    CU(cudaMemcpyAsync(host.data(), p->spectrum, host.size(), cudaMemcpyDeviceToHost, p->stream));
    CU(cudaStreamSynchronize(p->stream));
    const int kc = p->k_cut;
    for (int64_t i = 0; i < count; ++i) {
        int nx = modes[3 * i], ny = modes[3 * i + 1], nz = modes[3 * i + 2];
        const int s = nx * nx + ny * ny + nz * nz;
        bool in_k = s != 0 && s <= kc * kc;
        if (p->box) {
            // R26: |h|^2 Lmax^2 <= k_cut^2, the number fft_z_fused_kernel decides on (same products, same order)
            double lm = p->Lb[0] > p->Lb[1] ? p->Lb[0] : p->Lb[1];
            lm = lm > p->Lb[2] ? lm : p->Lb[2];
            const volatile double tx = (double)(nx * nx) * ((lm / p->Lb[0]) * (lm / p->Lb[0]));
            const volatile double ty = (double)(ny * ny) * ((lm / p->Lb[1]) * (lm / p->Lb[1]));
            const volatile double tz = (double)(nz * nz) * ((lm / p->Lb[2]) * (lm / p->Lb[2]));
            const volatile double txy = tx + ty;
            in_k = s != 0 && std::abs(nx) <= kc && std::abs(ny) <= kc && std::abs(nz) <= kc && txy + tz <= (double)(kc * kc);
        }
        if (!in_k) return fail(ENUF_EINVAL, "mode %lld is outside the cutoff set K (0 < |n|^2 <= k_cut^2)", (long long)i);
        const bool conj = nx < 0;            // S~(-n) = conj S~(n): only kx >= 0 is stored
        if (conj) { nx = -nx; ny = -ny; nz = -nz; }
        const int kyp = ny >= 0 ? ny : ny + p->Ky, kzp = nz >= 0 ? nz : nz + p->Ky;
        const size_t o = ((size_t)kzp * p->Ky + kyp) * p->Kxp + nx;
        double re, im;
        if (es == 4) { const float* h = reinterpret_cast<const float*>(host.data()); re = h[2 * o]; im = h[2 * o + 1]; }
        else { const double* h = reinterpret_cast<const double*>(host.data()); re = h[2 * o]; im = h[2 * o + 1]; }
        out[2 * i] = re;
        out[2 * i + 1] = conj ? -im : im;
    }
    return ENUF_OK;
}

int enuf_spread_only(enuf_plan* p, const void* r, const void* q, void* grid_host) {
    g_err[0] = 0;
    if (!p || !grid_host) return fail(ENUF_EINVAL, "plan or grid_host is NULL");
    if (p->N > 0 && (!r || !q)) return fail(ENUF_EINVAL, "r and q must be non-NULL when N > 0");
    int rc = prepare(p);
    if (rc) return rc;
    const size_t n = p->n, bytes = p->esize * n * n * n;
    p->launches = 0;
    if (p->N == 0) {
        CU(cudaMemsetAsync(p->grid[0], 0, bytes, p->stream));
    } else {
        // F of neutral particles is written by the bin kernel: use the staging-free scratch A1
        void* scratch = p->A1[0];
        if ((size_t)p->N * 3 * p->esize > 2 * p->esize * n * n * p->Kxp)
            return fail(ENUF_EINVAL, "enuf_spread_only: N too large for the scratch buffer");
        rc = p->precision == ENUF_F32 ? run_bin_spread<float>(p, r, q, scratch) : run_bin_spread<double>(p, r, q, scratch);
        if (rc) return fail_launch(p);
    }
    CU(cudaMemcpyAsync(grid_host, p->grid[0], bytes, cudaMemcpyDeviceToHost, p->stream));
    CU(cudaStreamSynchronize(p->stream));
    // scratch columns must be finite for later evaluations
    CU(cudaMemsetAsync(p->A1[0], 0, 2 * p->esize * n * n * p->Kxp, p->stream));
    return ENUF_OK;
}

void enuf_plan_destroy(enuf_plan* p) {
    if (!p) return;
    if (p->allocated) cudaStreamSynchronize(p->stream);
    free_workspace(p);
    if (p->cap_stream) cudaStreamDestroy(p->cap_stream);
    delete p;
}

int enuf_plan_create_auto(enuf_plan** out, int64_t N, double L, double delta, double r_c, double sigma, int m) {
    g_err[0] = 0;
    if (!out) return fail(ENUF_EINVAL, "out is NULL");
    *out = nullptr;
    if (!(delta > 0) || !(delta < 1)) return fail(ENUF_EINVAL, "delta must be in (0, 1)");
    if (!(r_c > 0) || !std::isfinite(r_c)) return fail(ENUF_EINVAL, "r_c must be positive and finite");
    if (!(L > 0) || !std::isfinite(L)) return fail(ENUF_EINVAL, "L must be positive and finite");
    const double alpha = std::sqrt(-std::log(delta)) / r_c;                                   // Eq. 32 (R15)
    const int k_cut = (int)std::ceil(alpha * L / kPi * std::sqrt(-std::log(delta)));          // Eq. 31 (R14)
    if (k_cut < 1 || k_cut > 4096) return fail(ENUF_EINVAL, "Eq. 31 gives k_cut = %d: out of range", k_cut);
    int M = 2;
    while (M < 2 * k_cut) M *= 2;                                                             // R5: k_cut <= M/2
    return enuf_plan_create(out, N, L, alpha, k_cut, M, sigma, m);
}

int enuf_plan_get(const enuf_plan* p, int key, double* value) {
    g_err[0] = 0;
    if (!p || !value) return fail(ENUF_EINVAL, "plan or value is NULL");
    switch (key) {
        case ENUF_GET_ALPHA: *value = p->alpha; return ENUF_OK;
        case ENUF_GET_K_CUT: *value = p->k_cut; return ENUF_OK;
        case ENUF_GET_M: *value = p->M; return ENUF_OK;
        case ENUF_GET_GRID: *value = p->n; return ENUF_OK;
        case ENUF_GET_SUPPORT: *value = p->m; return ENUF_OK;
        default: return fail(ENUF_EINVAL, "unknown key %d", key);
    }
}

int enuf_ncut(double alpha, double L, double delta) {
    if (!(alpha > 0) || !(L > 0) || !(delta > 0) || !(delta < 1)) return -1;
    return (int)std::ceil(alpha * L / kPi * std::sqrt(-std::log(delta)));
}

double enuf_alpha_from_rc(double r_c, double delta) {
    if (!(r_c > 0) || !(delta > 0) || !(delta < 1)) return NAN;
    return std::sqrt(-std::log(delta)) / r_c;
}

double enuf_rc_from_ncut(int n_c, double alpha, double L) {
    if (n_c < 1 || !(alpha > 0) || !(L > 0)) return NAN;
    return kPi * n_c / (alpha * alpha * L);
}

}  // extern "C"

// ====================================================================== allocation-free entry point
// enuf_self_energy_static (include/enuf.h): E_self = (alpha / sqrt(pi)) sum_i q_i^2 (Eq. 24), the
// quantity enuf_real_space returns as *E_self, for callers that must not allocate (CUDA graph capture, serving
// loops).  It is the two-level fp64 reduction of the real-space path (per-CTA partial sums, then one fixed-order
// final sum; enuf_real.cuh) with its scratch -- the partial sums and the count of finished CTAs -- in a file-scope
// device array instead of plan workspace.  Every GPU that loads the library holds the array (128.25 KiB) until exit.
// Every call shares it: calls that overlap on the GPU (two streams, two host threads) race; calls on one stream do not.
namespace {

constexpr int kSelfThreads = 256, kSelfPerCta = 4 * kSelfThreads;      // 1024 charges per CTA
constexpr int64_t kSelfMaxN = (int64_t)1 << 24;                        // ENUF_SELF_STATIC_MAX_N
constexpr int kSelfMaxCtas = (int)(kSelfMaxN / kSelfPerCta);           // 16384 partial sums
constexpr size_t kSelfCountOffset = sizeof(double) * kSelfMaxCtas;     // the finished-CTA counter follows the partials
static_assert(kSelfMaxN == ENUF_SELF_STATIC_MAX_N, "header and kernel limits differ");

static __device__ __align__(256) unsigned char g_self_scratch[kSelfCountOffset + 256];

// partial[b] = sum of q_i^2 over the CTA's 1024 charges (fp64; fp32 charges are promoted exactly).  The CTA that
// finishes last adds the partials in a fixed order (strided per thread, then a tree: the same whichever CTA it is)
// and writes out[0] = scale * sum.  *done must be 0 at launch (the host clears it on the stream before every launch).
template <typename T>
__global__ void __launch_bounds__(kSelfThreads)
self_energy_static_kernel(const T* __restrict__ q, int64_t N, double scale, double* __restrict__ partial,
                          unsigned* __restrict__ done, double* __restrict__ out) {
    __shared__ double red[kSelfThreads];
    __shared__ bool is_last;
    const int64_t base = (int64_t)blockIdx.x * kSelfPerCta;
    double s = 0.0;
#pragma unroll
    for (int k = 0; k < kSelfPerCta / kSelfThreads; ++k) {
        const int64_t i = base + (int64_t)k * kSelfThreads + threadIdx.x;
        if (i < N) { const double v = (double)q[i]; s += v * v; }
    }
    red[threadIdx.x] = s;
    __syncthreads();
    for (int o = kSelfThreads / 2; o > 0; o >>= 1) {
        if ((int)threadIdx.x < o) red[threadIdx.x] += red[threadIdx.x + o];
        __syncthreads();
    }
    if (threadIdx.x == 0) {
        partial[blockIdx.x] = red[0];
        __threadfence();
        is_last = atomicAdd(done, 1u) == gridDim.x - 1;
    }
    __syncthreads();
    if (!is_last) return;
    __threadfence();
    double t = 0.0;
    for (unsigned i = threadIdx.x; i < gridDim.x; i += kSelfThreads) t += __ldcg(&partial[i]);
    red[threadIdx.x] = t;
    __syncthreads();
    for (int o = kSelfThreads / 2; o > 0; o >>= 1) {
        if ((int)threadIdx.x < o) red[threadIdx.x] += red[threadIdx.x + o];
        __syncthreads();
    }
    if (threadIdx.x == 0) out[0] = scale * red[0];
}

// Device address of g_self_scratch on the current device.  In host code the array's name is only a handle:
// the address comes from cudaGetSymbolAddress, asked once per device with that device current.
constexpr int kSelfMaxDevices = 64;
void* g_self_addr[kSelfMaxDevices] = {nullptr};
int self_scratch_address(void** out) {
    int dev = 0;
    CU(cudaGetDevice(&dev));
    if (dev >= 0 && dev < kSelfMaxDevices) {
        void* cached = __atomic_load_n(&g_self_addr[dev], __ATOMIC_ACQUIRE);
        if (cached) { *out = cached; return ENUF_OK; }
    }
    void* ptr = nullptr;
    CU(cudaGetSymbolAddress(&ptr, g_self_scratch));
    if (!ptr) return fail(ENUF_ECUDA, "cudaGetSymbolAddress returned a null address");
    if (dev >= 0 && dev < kSelfMaxDevices) __atomic_store_n(&g_self_addr[dev], ptr, __ATOMIC_RELEASE);
    *out = ptr;
    return ENUF_OK;
}

}  // namespace

extern "C" int enuf_self_energy_static(const void* q, int64_t N, int precision, double alpha, void* cuda_stream,
                                       double* E_self) {
    g_err[0] = 0;
    if (!E_self) return fail(ENUF_EINVAL, "E_self is NULL");
    if (precision != ENUF_F32 && precision != ENUF_F64) return fail(ENUF_EINVAL, "precision must be ENUF_F32 or ENUF_F64");
    if (!(alpha > 0) || !std::isfinite(alpha)) return fail(ENUF_EINVAL, "alpha must be positive and finite");
    if (N < 0) return fail(ENUF_EINVAL, "N = %lld is negative", (long long)N);
    if (N > kSelfMaxN)
        return fail(ENUF_EINVAL, "N = %lld exceeds ENUF_SELF_STATIC_MAX_N = %lld, the size the static scratch array was "
                    "built for; use enuf_real_space", (long long)N, (long long)kSelfMaxN);
    if (N > 0 && !q) return fail(ENUF_EINVAL, "q must be non-NULL when N > 0");
    void* scratch = nullptr;
    int rc = self_scratch_address(&scratch);
    if (rc) return rc;
    cudaStream_t s = static_cast<cudaStream_t>(cuda_stream);
    double* partial = static_cast<double*>(scratch);
    unsigned* done = reinterpret_cast<unsigned*>(static_cast<unsigned char*>(scratch) + kSelfCountOffset);
    const unsigned ctas = N > 0 ? (unsigned)((N + kSelfPerCta - 1) / kSelfPerCta) : 1u;
    const double scale = alpha * 0.56418958354775628694807945156077;     // alpha / sqrt(pi)
    // the array keeps what the last call left: the counter must start at zero (the partials are overwritten)
    CU(cudaMemsetAsync(done, 0, sizeof(unsigned), s));
    if (precision == ENUF_F32)
        self_energy_static_kernel<float><<<ctas, kSelfThreads, 0, s>>>(static_cast<const float*>(q), N, scale, partial, done, E_self);
    else
        self_energy_static_kernel<double><<<ctas, kSelfThreads, 0, s>>>(static_cast<const double*>(q), N, scale, partial, done, E_self);
    CU(cudaGetLastError());
    return ENUF_OK;
}

// Host-only check of the spreading kernel's work decomposition (enuf_common.cuh: spread_split_make, spread_piece,
// spread_piece_start) for a grid, window and device size: every (column, plane) slab in exactly one piece, no piece
// shorter than the planes it shares with its neighbour, every piece start among the starts that are zeroed.
extern "C" int enuf_spread_split_check(int n, int m, int precision, int trimmed, int num_sms, int zchunk, int* G_out,
                                       int* min_slabs_out, int* max_slabs_out) {
    g_err[0] = 0;
    if (n < 32 || n > 1024 || n % 16 != 0) return fail(ENUF_EINVAL, "n = %d must be a multiple of 16 in [32, 1024]", n);
    if (m < 1 || m > enuf::kMaxM || num_sms < 1 || zchunk < 0 || zchunk > n) return fail(ENUF_EINVAL, "bad m, num_sms or zchunk");
    const int npx = n >= 128 ? 4 : 2;
    if (n % (8 * npx) != 0) return fail(ENUF_EINVAL, "n = %d is not a multiple of the column width %d", n, 8 * npx);
    const int per_sm = precision == ENUF_F32 ? enuf::spread_ctas_per_sm<float>(npx) : enuf::spread_ctas_per_sm<double>(npx);
    const enuf::SpreadSplit sp = enuf::spread_split_make(n, npx, m, trimmed != 0, (long long)num_sms * per_sm, zchunk);
    std::vector<unsigned char> cover((size_t)sp.ncol * n, 0);
    std::vector<unsigned char> zeroed((size_t)sp.ncol * n, 0);
    for (int i = 0; i < sp.G + sp.ncol; ++i) {
        int col, z0;
        if (enuf::spread_piece_start(sp, i, col, z0)) {
            if (col < 0 || col >= sp.ncol || z0 < 0 || z0 >= n) return fail(ENUF_EINVAL, "piece start %d out of range", i);
            zeroed[(size_t)col * n + z0] = 1;
        }
    }
    int lo = 1 << 30, hi = 0;
    for (int c = 0; c < sp.G; ++c) {
        int tot = 0;
        enuf::SpreadPiece pc;
        for (int i = 0; enuf::spread_piece(sp, c, i, pc); ++i) {
            if (pc.col < 0 || pc.col >= sp.ncol || pc.z0 < 0 || pc.z1 > n || pc.z0 >= pc.z1)
                return fail(ENUF_EINVAL, "CTA %d piece %d = (col %d, [%d, %d)) out of range", c, i, pc.col, pc.z0, pc.z1);
            if (zchunk == 0 && pc.z1 - pc.z0 < sp.minlen && pc.z1 - pc.z0 < n)
                return fail(ENUF_EINVAL, "CTA %d piece %d has %d planes, fewer than the %d it shares", c, i, pc.z1 - pc.z0, sp.minlen);
            if (!zeroed[(size_t)pc.col * n + pc.z0])
                return fail(ENUF_EINVAL, "start of CTA %d piece %d (col %d, z %d) is not zeroed", c, i, pc.col, pc.z0);
            for (int z = pc.z0; z < pc.z1; ++z)
                if (cover[(size_t)pc.col * n + z]++) return fail(ENUF_EINVAL, "slab (col %d, z %d) is in two pieces", pc.col, z);
            tot += pc.z1 - pc.z0;
        }
        if (tot > 0) { lo = tot < lo ? tot : lo; hi = tot > hi ? tot : hi; }
    }
    for (size_t i = 0; i < cover.size(); ++i)
        if (!cover[i]) return fail(ENUF_EINVAL, "slab (col %d, z %d) is in no piece", (int)(i / n), (int)(i % n));
    for (int col = 0; col < sp.ncol; ++col)     // a column's top wraps onto its first piece
        if (!zeroed[(size_t)col * n]) return fail(ENUF_EINVAL, "start of column %d is not zeroed", col);
    if (G_out) *G_out = sp.G;
    if (min_slabs_out) *min_slabs_out = lo;
    if (max_slabs_out) *max_slabs_out = hi;
    return ENUF_OK;
}
