// Shared declarations of the CUDA ENUF library (sm_100a).  Product code: shares nothing
// with oracle/.  Notation follows the paper / DESIGN.md: n = sigma*M grid points per
// dimension, m = window cut-off, W = 2m+1 stencil points, u = n*x grid coordinate,
// c = floor(u+1/2) nearest grid point, d0 = u - c in [-1/2, 1/2).
#pragma once

#include <cuda_runtime.h>
#include <stdint.h>

#include "../../include/enuf.h"

namespace enuf {

constexpr int kMaxM = 6;            // largest supported window cut-off
constexpr int kMaxW = 2 * kMaxM + 1;
constexpr int kErfcDeg = 10;        // degree of the fp32 erfc fit of the real-space pair term (enuf_real.cuh)
constexpr int kLinesPerGroup = 8;   // FFT: consecutive kx handled together (64 B of complex fp32)

template <typename T> struct Cx2;
template <> struct Cx2<float> { using type = float2; };
template <> struct Cx2<double> { using type = double2; };
template <typename T> using Cx = typename Cx2<T>::type;

template <typename T> struct Vec4;
template <> struct Vec4<float> { using type = float4; };
template <> struct Vec4<double> { using type = double4; };

// Window parameters, precomputed on the host in fp64 (step a0).
struct WindowParams {
    int kind;          // ENUF_WINDOW_*
    int m;
    double b;          // Gaussian: 2 sigma m/((2 sigma-1) pi); Kaiser-Bessel: pi (2 - 1/sigma); sinc-power: pi (2 - 1/sigma)/(2m)
    double inv_b;      // 1/b (Gaussian)
    double bm;         // b*m
    double inv1m;      // 1/(1 - exp(-2 b m))      (Kaiser-Bessel)
    double A;          // m / sinh(b m)            (Kaiser-Bessel)
};

// One binned particle: fractional offset d0 per dimension and charge.
template <typename T> struct alignas(4 * sizeof(T)) PRec { T dx, dy, dz, q; };
// The sorted particle array: record, packed nearest cell and caller index side by side, so that the
// scatter writes one 32-byte sector per particle (fp32) and the spreading cull, which first reads the
// cell and then -- for the particles it keeps -- the record, finds the record in the line it just fetched.
template <typename T> struct alignas(sizeof(T) == 4 ? 32 : 16) PSlot { PRec<T> rec; uint32_t cell, idx; };

// Geometry shared by bin / spread / gather.  Particles are counting-sorted into bins
//   bin = (Ty * n + bz) * nt + Tx,   Tx = cx / 16, Ty = cy / 16, bz = the particle's grid plane
// (a column of 16 x 16 cells in x, y; one grid plane in z; x-neighbouring columns adjacent), so that
//   - the particles of plane bz in a run of x-neighbouring columns are ONE contiguous range: the spreading
//     producer reads the halo of its column, slab by slab, as three such ranges (one per row of columns), and
//   - the particles of a 16^3 tile are 16 ranges, one per plane (gather).
constexpr int kTile = 16;
struct TileGeom {
    int n;        // grid points per dimension
    int nt;       // columns per dimension = n / 16
    int nbins;    // nt * nt * n
    int trim;     // 1: the z index of the bin is c_z - 1 + (d0_z > 0) instead of c_z (trimmed stencils,
                  //    fp32 Kaiser-Bessel m >= 5: the particle's 2m non-zero z weights sit on the planes
                  //    bin_z - m + 1 .. bin_z + m)
};

// Work decomposition of the spreading kernel (enuf_spread.cuh, header comment).  The ncol * n slabs (column, bin plane)
// are cut into PIECES (column, [z0, z1)) and every CTA gets about S / G slabs:
//   chunk > 0: fixed pieces of `chunk` planes, one per CTA, G = ncol * ceil(n / chunk) (ENUF_OPT_SPREAD_ZCHUNK);
//   chunk = 0: every column is cut at the SAME planes into q full pieces [cut(j), cut(j+1)), cut(j) = j zr0 / q, of about
//              S / G planes each -- CTA c < q ncol takes piece j = c / ncol of column c % ncol, so that these CTAs sweep
//              their columns in step and a particle in the halo of several columns is fetched by all of them at about
//              the same time (it is still in L2 for the later ones) -- and the remainders [zr0, n) of the columns, laid
//              end to end, are shared equally among the other G - q ncol CTAs (a range of them is a few pieces of
//              neighbouring columns).  q = 0 (fewer CTAs than columns): zr0 = 0, everything is "remainder".
//              A range boundary closer than `minlen` to the start of a column's remainder is moved onto it, so that no
//              piece is shorter than minlen = WZ - 1 planes: every grid plane then receives from at most two pieces and
//              the sum of the two reductions does not depend on their order.
struct SpreadSplit {
    int G, n, ncol, chunk, minlen;
    int q, zr0;
};
struct SpreadPiece { int col, z0, z1; };
// boundary b (0..Grem) of the remainder space: columns of rlen = n - zr0 planes laid end to end
__host__ __device__ inline int spread_rem_boundary(const SpreadSplit& sp, int b) {
    const int rlen = sp.n - sp.zr0, grem = sp.G - sp.q * sp.ncol;
    int u = (int)(((long long)b * sp.ncol * rlen) / grem);
    const int z = u % rlen;
    if (z != 0) {
        if (z < sp.minlen) u -= z;
        else if (rlen - z < sp.minlen) u += rlen - z;
    }
    return u;
}
// the i-th piece of CTA c; false when the CTA has fewer pieces
__host__ __device__ inline bool spread_piece(const SpreadSplit& sp, int c, int i, SpreadPiece& pc) {
    if (sp.chunk > 0) {
        if (i > 0) return false;
        const int cpc = (sp.n + sp.chunk - 1) / sp.chunk;
        pc.col = c / cpc;
        pc.z0 = (c - pc.col * cpc) * sp.chunk;
        pc.z1 = pc.z0 + sp.chunk < sp.n ? pc.z0 + sp.chunk : sp.n;
        return true;
    }
    if (c < sp.q * sp.ncol) {
        if (i > 0) return false;
        const int j = c / sp.ncol;
        pc.col = c - j * sp.ncol;
        pc.z0 = (int)(((long long)j * sp.zr0) / sp.q);
        pc.z1 = (int)(((long long)(j + 1) * sp.zr0) / sp.q);
        return true;
    }
    const int rlen = sp.n - sp.zr0, cr = c - sp.q * sp.ncol;
    const int ulo = spread_rem_boundary(sp, cr), uhi = spread_rem_boundary(sp, cr + 1);
    const int u = i == 0 ? ulo : (ulo / rlen + i) * rlen;      // later pieces start with their column's remainder
    if (u >= uhi) return false;
    pc.col = u / rlen;
    pc.z0 = sp.zr0 + (u - pc.col * rlen);
    pc.z1 = pc.z0 + (uhi - u) < sp.n ? pc.z0 + (uhi - u) : sp.n;
    return true;
}
// Where pieces start = where two pieces share planes (a piece ends where another starts, or at the top of its column,
// which wraps onto the column's first piece): start number i of the G + ncol that spread_zero_block clears.
//   i < q ncol: full piece i;  then ncol: the remainders' starts (col, zr0);  then G - q ncol: the remainder CTAs' first pieces.
__host__ __device__ inline bool spread_piece_start(const SpreadSplit& sp, int i, int& col, int& z0) {
    if (sp.chunk > 0) {
        if (i >= sp.G) return false;
        SpreadPiece pc;
        spread_piece(sp, i, 0, pc);
        col = pc.col; z0 = pc.z0;
        return true;
    }
    SpreadPiece pc;
    if (i < sp.q * sp.ncol) { spread_piece(sp, i, 0, pc); col = pc.col; z0 = pc.z0; return true; }
    i -= sp.q * sp.ncol;
    if (sp.zr0 >= sp.n) return false;                            // no remainders
    if (i < sp.ncol) { col = i; z0 = sp.zr0; return true; }
    i -= sp.ncol;
    if (i >= sp.G - sp.q * sp.ncol) return false;
    if (!spread_piece(sp, sp.q * sp.ncol + i, 0, pc)) return false;
    col = pc.col; z0 = pc.z0;
    return true;
}
// The decomposition for a grid of n points, columns of 8 npx x 16 cells, window cut-off m (trimmed stencils: 2m planes)
// on a device that holds `slots` spreading CTAs at once; zchunk > 0 asks for fixed pieces instead (host only).
// q full pieces per column, cut at the same planes in all columns; the other CTAs share the remainders [zr0, n), the
// remainders of k whole columns each (k the smallest divisor of ncol that the resident CTAs allow): with L slabs per
// CTA, q L + L / k = n, i.e. L = k n / (1 + k q) and G = q ncol + ncol / k.
inline SpreadSplit spread_split_make(int n, int npx, int m, bool trim, long long slots, int zchunk) {
    SpreadSplit sp{};
    sp.n = n;
    sp.ncol = (n / (8 * npx)) * (n / 16);
    sp.minlen = 2 * m - (trim ? 1 : 0);
    sp.q = 0; sp.zr0 = 0;
    if (zchunk > 0) {
        sp.chunk = zchunk;
        sp.G = sp.ncol * ((n + zchunk - 1) / zchunk);
        return sp;
    }
    sp.chunk = 0;
    const long long slabs = (long long)sp.ncol * n;
    long long G = slots;
    const long long gmax = slabs / (sp.minlen + 1);
    if (G > gmax) G = gmax;
    if (G < 1) G = 1;
    const double len = (double)slabs / (double)G;                 // slabs per CTA if G divided them exactly
    sp.q = (int)((double)n / len + 1e-9);
    if (sp.q > 0) {
        const double spare = (double)G / sp.ncol - sp.q;          // CTAs per column beyond the q full pieces
        int k = spare > 1e-9 ? (int)(1.0 / spare - 1e-9) + 1 : sp.ncol + 1;
        while (k <= sp.ncol && sp.ncol % k != 0) ++k;
        if (k <= sp.ncol) {
            const double L = (double)k * n / (1.0 + (double)k * sp.q);
            sp.zr0 = (int)(sp.q * L + 0.5);
            G = (long long)sp.q * sp.ncol + sp.ncol / k;
        }
        if (k > sp.ncol || sp.zr0 > n - sp.minlen) {              // no remainder worth a piece: q equal pieces per column
            sp.zr0 = n;
            G = (long long)sp.q * sp.ncol;
        }
    }
    sp.G = (int)G;
    return sp;
}
// Piecewise-polynomial window table for the fp32 path (step a0).  For every stencil offset
// j in [0, m] the weight phi(d0 - j), d0 in [-1/2, 1/2], is a polynomial p_j of degree
// poly_degree(m) in d0 (Chebyshev interpolant of the window's analytic continuation, fitted
// in fp64 on the host; max error <= 5e-11 of phi(0), <= 2e-9 of max|phi'| for the
// derivative); since phi is even, p_{-j}(d0) = p_j(-d0),
// so with p_j = E_j(d0^2) + d0 O_j(d0^2) both come out of one evaluation of E_j and O_j.
// dphi is the exact derivative of that polynomial.  The table is passed to the kernels BY
// VALUE as a __grid_constant__ parameter: with fully unrolled loops every coefficient is a
// constant-bank operand of an FFMA, so the W weights of a stencil cost ~6 W FFMAs, no loads.
__host__ __device__ constexpr int poly_degree(int m) { return m >= 4 ? 10 : 12; }
constexpr int kPolyMaxDeg = 12;
template <int M_>
struct PolyArg {
    static constexpr int D = poly_degree(M_);          // even
    float c[D + 1][M_ + 1];   // value:      p_j(d0)  = sum_i c[i][j] d0^i,  j = 0..m
    float d[D][M_ + 1];       // derivative: p_j'(d0) = sum_i d[i][j] d0^i
    // The same coefficients paired for the packed evaluation (stencil_weights<.., kPacked = true>):
    // p_j(d0) = E_j(y) + d0 O_j(y), y = d0^2; the two Horner chains advance together in one FFMA2 per step,
    // vp[k][j] = (c_(D-2-2k), c_(D-1-2k)), top[j] = c_D starts E_j one step early (it has one coefficient more);
    // p_j' (degree D-1, odd) has D/2 coefficients in both chains: dp[k][j] = (d_(D-2-2k), d_(D-1-2k)).
    static constexpr int NP = D / 2;
    alignas(8) float top[M_ + 1 + ((M_ + 1) & 1)];
    float2 vp[NP][M_ + 1];
    float2 dp[NP][M_ + 1];
    // B-spline window (order 2m): for d0 in [0, 1/2] the weight phi(d0 - j), j = -m..m, is ONE polynomial piece of
    // degree 2m - 1 in d0 (the knots are the integers), stored exactly: bc[i][j + m] t^i; bd = its derivative.
    // For d0 < 0 the evenness of phi gives w_j(d0) = w_{-j}(-d0).
    float bc[2 * M_][2 * M_ + 1];
    float bd[2 * M_][2 * M_ + 1];
};

__host__ __device__ inline int bin_index(const TileGeom& g, int tx, int ty, int bz) { return (ty * g.n + bz) * g.nt + tx; }

__host__ __device__ inline uint32_t pack_cell(int cx, int cy, int cz) {
    return (uint32_t)cx | ((uint32_t)cy << 10) | ((uint32_t)cz << 20);
}
__host__ __device__ inline void unpack_cell(uint32_t p, int& cx, int& cy, int& cz) {
    cx = p & 1023u; cy = (p >> 10) & 1023u; cz = (p >> 20) & 1023u;
}

// ---------------------------------------------------------------- programmatic dependent launch
// First statement of every hot-path kernel.  When the kernel was launched with the programmatic-stream-serialization
// attribute (enuf_launch.cuh, pdl_launch) its CTAs may be scheduled while the preceding kernel still runs: `wait` then
// blocks until that kernel has completed and its memory is visible, so nothing of this kernel's reads or writes moves
// ahead of it -- only the launch latency and the CTA start-up overlap.  `launch_dependents` lets the NEXT kernel in the
// stream do the same with this one; that kernel starts only once every CTA of this one has issued it (i.e. is resident
// or done), so a waiting dependent never keeps a CTA of this grid off the machine (the single-launch scan relies on
// all of its CTAs being resident).  Without the attribute both instructions are no-ops.
__device__ __forceinline__ void pdl_prologue() {
    asm volatile("griddepcontrol.launch_dependents;" ::: "memory");
    asm volatile("griddepcontrol.wait;" ::: "memory");
}

// ---------------------------------------------------------------- mbarrier (shared::cta) wrappers
// Box edges per direction (cubic: three times L).  Orthorhombic boxes keep ONE grid size n in all directions
// (R26); only x_d = r_d / L_d, the k-space weight and the force prefactors know the edges.
struct Edges { double l[3]; };

__device__ __forceinline__ uint32_t smem_u32(const void* p) { return (uint32_t)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void mbar_init(uint64_t* bar, uint32_t count) {
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(bar)), "r"(count) : "memory");
}
__device__ __forceinline__ void mbar_expect_tx(uint64_t* bar, uint32_t bytes) {
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(bar)), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_wait(uint64_t* bar, uint32_t parity) {
    asm volatile(
        "{\n"
        ".reg .pred p;\n"
        "WAIT_%=:\n"
        "mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n"
        "@p bra DONE_%=;\n"
        "bra WAIT_%=;\n"
        "DONE_%=:\n"
        "}\n" ::"r"(smem_u32(bar)), "r"(parity) : "memory");
}
// same for waits that can be long (another warp's work): sleep between tries, with a growing interval, instead of
// spinning through issue slots that the working warps of the SM need
__device__ __forceinline__ void mbar_wait_backoff(uint64_t* bar, uint32_t parity) {
    uint32_t done, ns = 32;
    for (;;) {
        asm volatile(
            "{\n"
            ".reg .pred p;\n"
            "mbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n"
            "selp.u32 %0, 1, 0, p;\n"
            "}\n" : "=r"(done) : "r"(smem_u32(bar)), "r"(parity) : "memory");
        if (done) break;
        __nanosleep(ns);
        ns = ns < 512u ? 2u * ns : ns;
    }
}
__device__ __forceinline__ void mbar_arrive(uint64_t* bar) {
    asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(smem_u32(bar)) : "memory");
}
// the same on a shared-window address the caller keeps (inner loops: no generic-to-shared conversion per call)
__device__ __forceinline__ void mbar_wait_backoff(uint32_t bar32, uint32_t parity) {
    uint32_t done, ns = 32;
    for (;;) {
        asm volatile(
            "{\n"
            ".reg .pred p;\n"
            "mbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n"
            "selp.u32 %0, 1, 0, p;\n"
            "}\n" : "=r"(done) : "r"(bar32), "r"(parity) : "memory");
        if (done) break;
        __nanosleep(ns);
        ns = ns < 512u ? 2u * ns : ns;
    }
}
__device__ __forceinline__ void mbar_arrive(uint32_t bar32) {
    asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(bar32) : "memory");
}

// ---------------------------------------------------------------- math wrappers
__device__ __forceinline__ float r_exp(float x) { return expf(x); }
__device__ __forceinline__ double r_exp(double x) { return exp(x); }
__device__ __forceinline__ float r_expm1(float x) { return expm1f(x); }
__device__ __forceinline__ double r_expm1(double x) { return expm1(x); }
__device__ __forceinline__ void r_sincos(float x, float* s, float* c) { sincosf(x, s, c); }
__device__ __forceinline__ void r_sincos(double x, double* s, double* c) { sincos(x, s, c); }
__device__ __forceinline__ float r_sqrt(float x) { return sqrtf(x); }
__device__ __forceinline__ double r_sqrt(double x) { return sqrt(x); }

// Window phi(d) and derivative phi'(d), d in grid units, phi(0) = 1 (R6, R7).
//   Gaussian:       phi = exp(-d^2/b)
//   Kaiser-Bessel:  phi = [sinh(b s)/s] * m/sinh(b m), s = sqrt(m^2 - d^2), 0 for |d| > m,
//                   evaluated overflow-free as (m/s) e^{b(s-m)} (1-e^{-2bs})/(1-e^{-2bm}).
//   sinc-power:     phi = sinc(t)^{2m}, t = b d, b = pi (2 - 1/sigma)/(2m);
//                   phi' = 2m sinc^{2m-1} b (t cos t - sin t)/t^2, the bracket by its series for |t| < 1/2.
//
// The stencil point is passed as (d0, j) with d = d0 - j, d0 = u - c in [-1/2, 1/2] and j the
// integer stencil offset.  d^2 is formed as j^2 + d0 (d0 - 2j) and the Kaiser-Bessel exponent
// b (s - m) as -b d^2/(s + m): in fp32 the direct forms lose ~ulp(m) = 5e-7 in s - m, i.e. a
// relative error of b*5e-7 = 2e-6 on the CENTRAL weights (fp32 error budget).
// Centred cardinal B-spline of order P and its derivative (de Boor's triangle on uniform knots; all terms positive).
// M_k(t) on [0, k], t = x + P/2:  M_k(t - j) = [(t - j) M_{k-1}(t - j) + (k - t + j) M_{k-1}(t - j - 1)] / (k - 1),
// M_P'(t) = M_{P-1}(t) - M_{P-1}(t - 1).
template <typename T, int P>
__host__ __device__ inline void bspline_eval(T x, T& val, T& dval) {
    const T t = x + (T)(0.5 * P);
    val = (T)0; dval = (T)0;
    if (!(t > (T)0) || !(t < (T)P)) return;
    T a[P + 1];
    const int i0 = (int)t;
#pragma unroll
    for (int j = 0; j <= P; ++j) a[j] = j == i0 ? (T)1 : (T)0;
    if (P == 2) dval = a[0] - a[1];
#pragma unroll
    for (int k = 2; k <= P; ++k) {
#pragma unroll
        for (int j = 0; j + k <= P; ++j) a[j] = ((t - (T)j) * a[j] + ((T)k - t + (T)j) * a[j + 1]) / (T)(k - 1);
        if (k == P - 1) dval = a[0] - a[1];
    }
    val = a[0];
}

template <typename T, bool kDeriv, int M_ = 0>
__device__ __forceinline__ void window_eval(const WindowParams& wp, T d0, int j, T& phi, T& dphi) {
    const T jf = (T)j;
    const T d = d0 - jf;
    const T d2 = d0 * (d0 - (T)2 * jf) + jf * jf;
    if (wp.kind == ENUF_WINDOW_SINC_POWER) {
        if constexpr (M_ > 0) {
            const T pc = (T)wp.b, t = pc * d, t2 = t * t;
            T sn, cs;
            r_sincos(t, &sn, &cs);
            const T sc = t == (T)0 ? (T)1 : sn / t;
            T pw = sc;                               // sinc^(2m-1)
#pragma unroll
            for (int i = 1; i < 2 * M_ - 1; ++i) pw *= sc;
            phi = pw * sc;
            if (kDeriv) {
                T g;                                 // (t cos t - sin t)/t^2 = -t/3 + t^3/30 - t^5/840 + ..
                if (t2 < (T)0.25)
                    g = -t * ((T)(1.0 / 3.0) - t2 * ((T)(1.0 / 30.0) - t2 * ((T)(1.0 / 840.0) - t2 * ((T)(1.0 / 45360.0)
                        - t2 * ((T)(1.0 / 3991680.0) - t2 * ((T)(1.0 / 518918400.0) - t2 * (T)(1.0 / 93405312000.0)))))));
                else
                    g = (t * cs - sn) / t2;
                dphi = (T)(2 * M_) * pw * pc * g;
            }
        }
    } else if (wp.kind == ENUF_WINDOW_BSPLINE) {
        if constexpr (M_ > 0) {
            T v, dv;
            bspline_eval<T, 2 * M_>(d, v, dv);
            phi = v * (T)wp.A;                       // A = 1 / B_2m(0)
            if (kDeriv) dphi = dv * (T)wp.A;
        }
    } else if (wp.kind == ENUF_WINDOW_GAUSSIAN) {
        T ib = (T)wp.inv_b;
        phi = r_exp(-d2 * ib);
        if (kDeriv) dphi = -(T)2 * d * ib * phi;
    } else {
        T m = (T)wp.m, b = (T)wp.b;
        T s2 = (m - d) * (m + d);
        if (s2 > (T)0) {
            T s = r_sqrt(s2);
            T e1 = r_exp(-b * d2 / (s + m));
            T e2m1 = r_expm1(-(T)2 * b * s);            // e^{-2bs} - 1
            T G = m * e1 * (T)wp.inv1m;                  // A e^{bs} / 2 ... scaled
            phi = -G * e2m1 / s;
            if (kDeriv) {
                T x = b * s;
                if (x < (T)1) {
                    T x2 = x * x;
                    // (x cosh x - sinh x)/x^3 = sum_{k>=1} 2k/(2k+1)! x^(2k-2); 8 terms: 1.5e-16 at x = 1
                    T ser = (T)(1.0 / 3.0) + x2 * ((T)(1.0 / 30.0) + x2 * ((T)(1.0 / 840.0)
                            + x2 * ((T)(1.0 / 45360.0) + x2 * ((T)(1.0 / 3991680.0)
                            + x2 * ((T)(1.0 / 518918400.0) + x2 * ((T)(1.0 / 93405312000.0)
                            + x2 * (T)(1.0 / 22230464256000.0)))))));
                    dphi = -(T)wp.A * d * b * b * b * ser;
                } else {
                    // -d G [b (1+e2) - (1-e2)/s] / s^2
                    dphi = -d * G * (b * ((T)2 + e2m1) + e2m1 / s) / s2;
                }
            }
        } else {
            phi = (s2 == (T)0) ? (T)(wp.A * wp.b) : (T)0;
            if (kDeriv) dphi = (T)0;
        }
    }
}


// All W = 2m+1 window weights (and derivatives) of one particle in one dimension:
//   w[k] = phi(d0 - (k - m)),  dw[k] = phi'(d0 - (k - m)),  k = 0..W-1.
//   fp32: the plan's polynomial table (even/odd Horner in d0^2); Kaiser-Bessel support cut
//         |d| <= m (value) and |d| < m (derivative) exactly as in the closed form.
//   fp64: the closed form (window_eval).
template <typename T, int M_, bool kDeriv, bool kPacked = false>
__device__ __forceinline__ void stencil_weights(const WindowParams& wp, const PolyArg<M_>& pa, T d0,
                                                T (&w)[2 * M_ + 1], T (&dw)[2 * M_ + 1]) {
    constexpr int W = 2 * M_ + 1;
    if (sizeof(T) == 8) {
#pragma unroll
        for (int k = 0; k < W; ++k) {
            dw[k] = (T)0;
            window_eval<T, kDeriv, M_>(wp, d0, k - M_, w[k], dw[k]);
        }
    } else {
        const float x = (float)d0, y = x * x;
        float v[W], dv[W];
        if (wp.kind == ENUF_WINDOW_BSPLINE) {
            // one exact polynomial piece per stencil offset on d0 in [0, 1/2]; d0 < 0 by symmetry
            const float t = fabsf(x);
            float u[W], du[W];
#pragma unroll
            for (int jj = 0; jj < W; ++jj) {
                float s = pa.bc[2 * M_ - 1][jj];
#pragma unroll
                for (int i = 2 * M_ - 2; i >= 0; --i) s = fmaf(s, t, pa.bc[i][jj]);
                u[jj] = s;
                float ds = 0.f;
                if (kDeriv) {
                    ds = pa.bd[2 * M_ - 2][jj];
#pragma unroll
                    for (int i = 2 * M_ - 3; i >= 0; --i) ds = fmaf(ds, t, pa.bd[i][jj]);
                }
                du[jj] = ds;
            }
            const bool neg = x < 0.f;
#pragma unroll
            for (int k = 0; k < W; ++k) { w[k] = (T)(neg ? u[W - 1 - k] : u[k]); dw[k] = (T)(neg ? -du[W - 1 - k] : du[k]); }
            return;
        }
        if constexpr (kPacked) {
            const float2 yy = make_float2(y, y);
            constexpr int NP = PolyArg<M_>::NP;
            {
                float2 EO[M_ + 1];                                     // (E_j, O_j)
#pragma unroll
                for (int j = 0; j <= M_; ++j) {
                    EO[j] = pa.vp[0][j];
                    EO[j].x = fmaf(pa.top[j], y, EO[j].x);
                }
#pragma unroll
                for (int k = 1; k < NP; ++k)
#pragma unroll
                    for (int j = 0; j <= M_; ++j) EO[j] = __ffma2_rn(EO[j], yy, pa.vp[k][j]);
                v[M_] = EO[0].x;                                       // p_0 is even
#pragma unroll
                for (int j = 1; j <= M_; ++j) { v[M_ + j] = fmaf(x, EO[j].y, EO[j].x); v[M_ - j] = fmaf(-x, EO[j].y, EO[j].x); }
            }
            if (kDeriv) {
                float2 EO[M_ + 1];                                     // (E'_j, O'_j) of p_j'
#pragma unroll
                for (int j = 0; j <= M_; ++j) EO[j] = pa.dp[0][j];
#pragma unroll
                for (int k = 1; k < NP; ++k)
#pragma unroll
                    for (int j = 0; j <= M_; ++j) EO[j] = __ffma2_rn(EO[j], yy, pa.dp[k][j]);
                dv[M_] = x * EO[0].y;                                  // p_0 is even: p_0' is odd
#pragma unroll
                for (int j = 1; j <= M_; ++j) { dv[M_ + j] = fmaf(x, EO[j].y, EO[j].x); dv[M_ - j] = fmaf(x, EO[j].y, -EO[j].x); }
            } else {
#pragma unroll
                for (int j = 0; j < W; ++j) dv[j] = 0.f;
            }
        } else {
            constexpr int D = PolyArg<M_>::D;
            constexpr int DE = D - (D & 1), DO = D - 1 + (D & 1);      // highest even / odd power of p
            {
                float E[M_ + 1], O[M_ + 1];
#pragma unroll
                for (int j = 0; j <= M_; ++j) { E[j] = pa.c[DE][j]; O[j] = pa.c[DO][j]; }
#pragma unroll
                for (int i = DE - 2; i >= 0; i -= 2)
#pragma unroll
                    for (int j = 0; j <= M_; ++j) E[j] = fmaf(E[j], y, pa.c[i][j]);
#pragma unroll
                for (int i = DO - 2; i >= 1; i -= 2)
#pragma unroll
                    for (int j = 1; j <= M_; ++j) O[j] = fmaf(O[j], y, pa.c[i][j]);
                v[M_] = E[0];
#pragma unroll
                for (int j = 1; j <= M_; ++j) { v[M_ + j] = fmaf(x, O[j], E[j]); v[M_ - j] = fmaf(-x, O[j], E[j]); }
            }
            if (kDeriv) {
                constexpr int D1 = D - 1;
                constexpr int DE1 = D1 - (D1 & 1), DO1 = D1 - 1 + (D1 & 1);
                float E[M_ + 1], O[M_ + 1];
#pragma unroll
                for (int j = 0; j <= M_; ++j) { E[j] = pa.d[DE1][j]; O[j] = pa.d[DO1][j]; }
#pragma unroll
                for (int i = DE1 - 2; i >= 0; i -= 2)
#pragma unroll
                    for (int j = 1; j <= M_; ++j) E[j] = fmaf(E[j], y, pa.d[i][j]);
#pragma unroll
                for (int i = DO1 - 2; i >= 1; i -= 2)
#pragma unroll
                    for (int j = 0; j <= M_; ++j) O[j] = fmaf(O[j], y, pa.d[i][j]);
                dv[M_] = x * O[0];                                       // p_0 is even: p_0' is odd
#pragma unroll
                for (int j = 1; j <= M_; ++j) { dv[M_ + j] = fmaf(x, O[j], E[j]); dv[M_ - j] = fmaf(x, O[j], -E[j]); }
            } else {
#pragma unroll
                for (int j = 0; j < W; ++j) dv[j] = 0.f;
            }
        }
        if (wp.kind == ENUF_WINDOW_KAISER_BESSEL) {
            // |d0 - j| > m only for j = +m (d0 < 0) and j = -m (d0 > 0); phi' = 0 at |d| = m
            if (x < 0.f) { v[W - 1] = 0.f; dv[W - 1] = 0.f; }
            if (x > 0.f) { v[0] = 0.f; dv[0] = 0.f; }
            if (x == 0.f) { dv[0] = 0.f; dv[W - 1] = 0.f; }
        }
#pragma unroll
        for (int j = 0; j < W; ++j) { w[j] = (T)v[j]; dw[j] = (T)dv[j]; }
    }
}

}  // namespace enuf
