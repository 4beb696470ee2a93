/*
 * enuf_oracle.c -- TEST INFRASTRUCTURE, NOT THE PRODUCT.
 *
 * Plain, slow, fp64 CPU implementation of what the ENUF reciprocal-space path
 * computes, written from the paper (arxiv 2004.12484, /root/reference/PAPER.md;
 * citations are PAPER.md:<line>) and from the readings listed in DESIGN.md /
 * SURVEY.md section 8(c) (R-numbers).  Only tests/, __graft_entry__.smoke() and bench.py's
 * cpu_baseline / --impl reference legs may call it.  It shares no code, header,
 * table or constant generator with the CUDA library under paper_2004_12484_b200/.
 *
 *   Oracle A  (orc_direct_*)  the definition: direct O(N*|K|) Ewald k-space sum,
 *             Eq. 37, Eq. 38 (:310), Eq. 41 (:332-336).
 *   Oracle B  (orc_spread / orc_fft3d / orc_scale / orc_gather, composed by
 *             orc_enuf)  the ENUF approximation, step by step in the paper's order
 *             (PAPER.md:491-499 spreading / FFT / scaling, subdividing / inverse FFT /
 *             interpolating), both force variants.
 *   Helpers   real-space + self energy (Eq. 17, 24, 25) used
 *             by the Madelung / Wigner pins; the parameter rule Eq. 31-32 (:256-259).
 *   Oracle R  (orc_real_forces)  the real-space part of the Ewald sum, energy per particle
 *             and forces (Eq. 16-17, 29) with the Slater factors
 *             B_U, B_F of Eq. 57-58 (:434-436); pinned by finite differences of the
 *             Madelung-pinned orc_real_energy, Newton's third law, Eq. 59-60 limits.
 *
 * Pins (tests/test_oracle_pins.py): rock-salt Madelung constant, cubic Wigner constant,
 * alpha-independence of the total energy, forces = -dE/dr by central differences,
 * sum_i F_i = 0, two-particle antisymmetry, window transform by quadrature, window
 * derivative by differences, DFT == radix-2 FFT == numpy.fft, additivity Eq. 61,
 * S~(n) vs S(n) mode by mode, error falls with m; B-spline window: m = 1 hat
 * function in closed form, partition of unity, transform by quadrature, derivative by differences,
 * brute force against Oracle A; sinc-power window (:266): transform by quadrature over the real line,
 * m = 1 transform = the textbook triangle, derivative by differences (both branches), brute force against Oracle A.
 * Parity unpinned against the paper: the Slater form factor in k-space (R19) -- it is
 * BASELINE.json's variant, pinned only against quadrature of Eq. 51 and Oracle A.
 *
 * Units: C = 1/(4 pi eps0) = 1, eps_r = 1 (R1).  Layout: r is N x 3 row-major,
 * grids are n x n x n with index (lz*n + ly)*n + lx (x fastest).
 * OpenMP pragmas sit only on loops whose iterations are independent.
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

#define ORC_PI 3.14159265358979323846264338327950288

enum { ORC_WIN_GAUSSIAN = 0, ORC_WIN_KAISER_BESSEL = 1, ORC_WIN_BSPLINE = 2, ORC_WIN_SINC_POWER = 3 };
enum { ORC_FORCE_ANALYTIC = 0, ORC_FORCE_IK = 1 };

int orc_num_threads(void)
{
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}

void orc_set_threads(int t)
{
#ifdef _OPENMP
    if (t > 0) omp_set_num_threads(t);
#else
    (void)t;
#endif
}

/* ------------------------------------------------------------------ windows
 * The paper names the windows and uses the Gaussian of Greengard-Lee
 * in CU-NFFT (:491, :499) but prints no formula; R6/R7: the NFFT-literature forms,
 * normalised to phi(0) = 1, argument d in grid units.                          */

static double gauss_b(int m, double sigma)
{
    return 2.0 * sigma * m / ((2.0 * sigma - 1.0) * ORC_PI);
}

static double kb_b(double sigma)
{
    return ORC_PI * (2.0 - 1.0 / sigma);
}

/* Centred cardinal B-spline of order p (degree p - 1, support [-p/2, p/2]) by its defining recursion
 * (Cox-de Boor for uniform knots): B_1 = indicator of [-1/2, 1/2),
 * B_p(x) = [(x + p/2) B_{p-1}(x + 1/2) + (p/2 - x) B_{p-1}(x - 1/2)] / (p - 1).
 * Slow (2^p leaves) and obviously the definition.  PAPER.md:266 names the B-spline among the NFFT
 * windows without a formula; the NFFT literature it cites uses order 2m, normalised here to phi(0) = 1 (R7). */
static double bspline_rec(int p, double x)
{
    if (p == 1) return (x >= -0.5 && x < 0.5) ? 1.0 : 0.0;
    return ((x + 0.5 * p) * bspline_rec(p - 1, x + 0.5) + (0.5 * p - x) * bspline_rec(p - 1, x - 0.5)) / (p - 1);
}

/* Sinc-power window (PAPER.md:266 names "sinc power functions" among the NFFT windows without a formula; the NFFT
 * literature it cites has phi(x) ~ sinc^{2m}(pi N x (2 sigma - 1)/(2m)), whose transform is a B-spline of order 2m).
 * With x = d/n, n = sigma N, and phi(0) = 1 (R7):
 *     phi(d) = sinc(pi c d)^{2m},  c = (2 - 1/sigma)/(2m),  sinc(t) = sin(t)/t;
 * sinc(pi c d) is the transform of a box of width c and height 1/c, so phi is the transform of the 2m-fold
 * convolution of that box:  Phi(k) = (1/c) B_2m(k/(n c)),  B_2m the centred cardinal B-spline of order 2m.
 * The window is not compactly supported; the stencil cuts it (R8), as it cuts the Gaussian. */
static double sincpow_c(int m, double sigma)
{
    return (2.0 - 1.0 / sigma) / (2.0 * m);
}

double orc_phi(int window, int m, double sigma, double d)
{
    if (window == ORC_WIN_SINC_POWER) {
        double t = ORC_PI * sincpow_c(m, sigma) * d;
        double sc = t == 0.0 ? 1.0 : sin(t) / t;
        return pow(sc, 2 * m);
    } else if (window == ORC_WIN_BSPLINE) {
        return bspline_rec(2 * m, d) / bspline_rec(2 * m, 0.0);
    } else if (window == ORC_WIN_GAUSSIAN) {
        return exp(-d * d / gauss_b(m, sigma));
    } else {
        double b = kb_b(sigma);
        double s2 = (double)m * m - d * d;
        double A = m / sinh(b * m);
        if (s2 > 0.0) {
            double s = sqrt(s2);
            return A * sinh(b * s) / s;
        }
        if (s2 == 0.0) return A * b;
        return 0.0;
    }
}

/* d phi / d d (used by the analytic-derivative force variant). */
double orc_dphi(int window, int m, double sigma, double d)
{
    if (window == ORC_WIN_SINC_POWER) {
        /* d/dd sinc(t)^{2m} = 2m sinc^{2m-1} pi c (t cos t - sin t)/t^2, t = pi c d;
         * (t cos t - sin t)/t^2 = sum_{k>=1} (-1)^k 2k/(2k+1)! t^(2k-1) without the cancellation for small t */
        double pc = ORC_PI * sincpow_c(m, sigma), t = pc * d, g, sc;
        if (fabs(t) < 0.5) {
            double t2 = t * t;
            g = -t * (1.0 / 3.0 - t2 * (1.0 / 30.0 - t2 * (1.0 / 840.0 - t2 * (1.0 / 45360.0
                - t2 * (1.0 / 3991680.0 - t2 * (1.0 / 518918400.0 - t2 / 93405312000.0))))));
            sc = t == 0.0 ? 1.0 : sin(t) / t;
        } else {
            g = (t * cos(t) - sin(t)) / (t * t);
            sc = sin(t) / t;
        }
        return 2.0 * m * pow(sc, 2 * m - 1) * pc * g;
    } else if (window == ORC_WIN_BSPLINE) {
        /* B_p' (x) = B_{p-1}(x + 1/2) - B_{p-1}(x - 1/2) */
        return (bspline_rec(2 * m - 1, d + 0.5) - bspline_rec(2 * m - 1, d - 0.5)) / bspline_rec(2 * m, 0.0);
    } else if (window == ORC_WIN_GAUSSIAN) {
        double b = gauss_b(m, sigma);
        return -(2.0 * d / b) * exp(-d * d / b);
    } else {
        double b = kb_b(sigma);
        double s2 = (double)m * m - d * d;
        double A = m / sinh(b * m);
        if (s2 <= 0.0) return 0.0;
        double s = sqrt(s2), x = b * s, bracket_over_s2;
        if (x < 0.25) {
            /* [b cosh x - b sinh x / x] / s^2 = b^3 sum_k x^(2k-2) 2k/(2k+1)! */
            double x2 = x * x;
            bracket_over_s2 = b * b * b * (1.0 / 3.0 + x2 * (1.0 / 30.0 + x2 * (1.0 / 840.0
                              + x2 * (1.0 / 45360.0 + x2 / 3991680.0))));
        } else {
            bracket_over_s2 = (b * cosh(x) - sinh(x) / s) / s2;
        }
        return -A * d * bracket_over_s2;
    }
}

/* modified Bessel function I0 by its power series sum_k ((x/2)^k / k!)^2 */
static double bessel_i0(double x)
{
    double h = 0.5 * x, term = 1.0, sum = 1.0;
    for (int k = 1; k < 500; ++k) {
        term *= (h / k) * (h / k);
        sum += term;
        if (term < 1e-17 * sum) break;
    }
    return sum;
}

/* Continuous Fourier transform of phi at the integer frequency k of an n-point grid:
 * Phi(k) = int phi(d) exp(-2 pi i k d / n) dd.                                   */
double orc_Phi(int window, int m, double sigma, int n, int k)
{
    if (window == ORC_WIN_SINC_POWER) {
        double c = sincpow_c(m, sigma);
        return bspline_rec(2 * m, (double)k / (n * c)) / c;
    } else if (window == ORC_WIN_BSPLINE) {
        /* B_p is the p-fold convolution of the unit box, whose transform at frequency k/n is sinc(pi k/n) */
        double t = ORC_PI * k / n, sc = k == 0 ? 1.0 : sin(t) / t;
        return pow(sc, 2 * m) / bspline_rec(2 * m, 0.0);
    } else if (window == ORC_WIN_GAUSSIAN) {
        double b = gauss_b(m, sigma);
        double t = ORC_PI * k / n;
        return sqrt(ORC_PI * b) * exp(-b * t * t);
    } else {
        double b = kb_b(sigma);
        double w = 2.0 * ORC_PI * k / n;
        double arg2 = b * b - w * w;
        double A = m / sinh(b * m);
        if (arg2 >= 0.0) return ORC_PI * A * bessel_i0(m * sqrt(arg2));
        /* beyond the pass band I0(i y) = J0(y); never reached for |k| <= n/(2 sigma) */
        return ORC_PI * A * j0(m * sqrt(-arg2));
    }
}

/* ------------------------------------------------------- Ewald k-space kernel */

/* w(n) of Eq. 38: exp(-(pi n)^2/(alpha L)^2) / n^2, n2 = |n|^2 integer */
double orc_w(int n2, double alpha, double L)
{
    double a = ORC_PI / (alpha * L);
    return exp(-a * a * n2) / n2;
}

/* R19: squared Fourier form factor of the Slater density Eq. 51,
 * f(k) = (1 + k^2 lambda^2/4)^-2 with k = 2 pi |n| / L; lambda = 0 -> point charge. */
double orc_slater_f2(int n2, double lambda, double L)
{
    if (lambda == 0.0) return 1.0;
    double t = ORC_PI * lambda / L;
    double g = 1.0 + t * t * n2;
    return 1.0 / (g * g * g * g);
}

/* Eq. 31: smallest integer n_c >= (alpha L/pi) sqrt(-ln delta) (R14) */
int orc_ncut(double alpha, double L, double delta)
{
    return (int)ceil(alpha * L / ORC_PI * sqrt(-log(delta)));
}

/* Eq. 32 read as alpha r_c = sqrt(-ln delta) (R15) */
double orc_alpha_from_rc(double r_c, double delta)
{
    return sqrt(-log(delta)) / r_c;
}

/* ------------------------------------------------------------------ Oracle A */

static double frac_pos(double r, double L)
{
    double x = r / L;          /* x = r/L */
    x -= floor(x);             /* R10 */
    if (x >= 1.0) x = 0.0;
    return x;
}

/* S(n) = sum_j q_j exp(-2 pi i n.x_j), Eq. 37, for a list of modes. */
void orc_direct_S(int64_t N, const double *r, const double *q, double L,
                  int64_t nmodes, const int *modes, double *S_re, double *S_im)
{
    double *x = (double *)malloc(sizeof(double) * 3 * (size_t)(N > 0 ? N : 1));
    for (int64_t j = 0; j < 3 * N; ++j) x[j] = frac_pos(r[j], L);
#pragma omp parallel for schedule(static)
    for (int64_t t = 0; t < nmodes; ++t) {
        double sr = 0.0, si = 0.0;
        int nx = modes[3 * t], ny = modes[3 * t + 1], nz = modes[3 * t + 2];
        for (int64_t j = 0; j < N; ++j) {
            double ph = 2.0 * ORC_PI * (nx * x[3 * j] + ny * x[3 * j + 1] + nz * x[3 * j + 2]);
            sr += q[j] * cos(ph);
            si -= q[j] * sin(ph);
        }
        S_re[t] = sr;
        S_im[t] = si;
    }
    free(x);
}

/* Enumerate K = { n : 0 < |n|^2 <= k_cut^2 } (R4, R12). Returns the count; fills modes
 * (3 ints each) if modes != NULL. */
int64_t orc_modes(int k_cut, int *modes)
{
    int64_t c = 0;
    for (int nz = -k_cut; nz <= k_cut; ++nz)
        for (int ny = -k_cut; ny <= k_cut; ++ny)
            for (int nx = -k_cut; nx <= k_cut; ++nx) {
                int n2 = nx * nx + ny * ny + nz * nz;
                if (n2 == 0 || n2 > k_cut * k_cut) continue;
                if (modes) { modes[3 * c] = nx; modes[3 * c + 1] = ny; modes[3 * c + 2] = nz; }
                ++c;
            }
    return c;
}

/* E_rec = (1/(2 pi L)) sum_K f^2 w |S|^2           Eq. 38
 * F_i   = (2 q_i/L^2) sum_K n f^2 w Im{S e^{+2 pi i n.x_i}}   Eq. 41
 * F may be NULL. If nsample > 0 only particles sample[0..nsample) get forces, written
 * to F[3*s]; otherwise all N.  Returns 0, or -1 on allocation failure.            */
int orc_direct(int64_t N, const double *r, const double *q, double L, double alpha,
               int k_cut, double lambda, double *E, double *F,
               int64_t nsample, const int64_t *sample)
{
    int64_t nK = orc_modes(k_cut, NULL);
    int *modes = (int *)malloc(sizeof(int) * 3 * (size_t)nK);
    double *Sr = (double *)malloc(sizeof(double) * (size_t)nK);
    double *Si = (double *)malloc(sizeof(double) * (size_t)nK);
    if (!modes || !Sr || !Si) { free(modes); free(Sr); free(Si); return -1; }
    orc_modes(k_cut, modes);
    orc_direct_S(N, r, q, L, nK, modes, Sr, Si);

    double e = 0.0;
    for (int64_t t = 0; t < nK; ++t) {
        int n2 = modes[3 * t] * modes[3 * t] + modes[3 * t + 1] * modes[3 * t + 1]
                 + modes[3 * t + 2] * modes[3 * t + 2];
        e += orc_slater_f2(n2, lambda, L) * orc_w(n2, alpha, L) * (Sr[t] * Sr[t] + Si[t] * Si[t]);
    }
    *E = e / (2.0 * ORC_PI * L);

    if (F) {
        int64_t nf = nsample > 0 ? nsample : N;
#pragma omp parallel for schedule(static)
        for (int64_t s = 0; s < nf; ++s) {
            int64_t i = nsample > 0 ? sample[s] : s;
            double xi = frac_pos(r[3 * i], L), yi = frac_pos(r[3 * i + 1], L), zi = frac_pos(r[3 * i + 2], L);
            double fx = 0.0, fy = 0.0, fz = 0.0;
            for (int64_t t = 0; t < nK; ++t) {
                int nx = modes[3 * t], ny = modes[3 * t + 1], nz = modes[3 * t + 2];
                int n2 = nx * nx + ny * ny + nz * nz;
                double ph = 2.0 * ORC_PI * (nx * xi + ny * yi + nz * zi);
                /* Im{ (Sr + i Si)(cos + i sin) } */
                double im = Sr[t] * sin(ph) + Si[t] * cos(ph);
                double c = orc_slater_f2(n2, lambda, L) * orc_w(n2, alpha, L) * im;
                fx += nx * c; fy += ny * c; fz += nz * c;
            }
            double pre = 2.0 * q[i] / (L * L);
            F[3 * s] = pre * fx; F[3 * s + 1] = pre * fy; F[3 * s + 2] = pre * fz;
        }
    }
    free(modes); free(Sr); free(Si);
    return 0;
}

/* ------------------------------------- real-space and self terms (pins only) */

/* (1/2) sum_i sum_j sum_images' q_i q_j erfc(alpha r)/r, r <= r_cut, image shells
 * |n_t| <= shells; the prime drops i = j in the home cell only (Eq. 1, 16: PAPER.md:93,
 * :176).                                                                         */
double orc_real_energy(int64_t N, const double *r, const double *q, double L, double alpha,
                       double r_cut, int shells)
{
    double e = 0.0;
#pragma omp parallel for schedule(dynamic, 16) reduction(+ : e)
    for (int64_t i = 0; i < N; ++i) {
        double ei = 0.0;
        for (int64_t j = 0; j < N; ++j)
            for (int a = -shells; a <= shells; ++a)
                for (int b = -shells; b <= shells; ++b)
                    for (int c = -shells; c <= shells; ++c) {
                        if (i == j && a == 0 && b == 0 && c == 0) continue;
                        double dx = r[3 * j] - r[3 * i] + a * L;
                        double dy = r[3 * j + 1] - r[3 * i + 1] + b * L;
                        double dz = r[3 * j + 2] - r[3 * i + 2] + c * L;
                        double d2 = dx * dx + dy * dy + dz * dz;
                        if (d2 > r_cut * r_cut) continue;
                        double d = sqrt(d2);
                        ei += q[i] * q[j] * erfc(alpha * d) / d;
                    }
        e += ei;
    }
    return 0.5 * e;
}

/* (alpha/sqrt(pi)) sum q_i^2, Eq. 24; subtracted in Eq. 25 (:223, R13) */
double orc_self_energy(int64_t N, const double *q, double alpha)
{
    double s = 0.0;
    for (int64_t i = 0; i < N; ++i) s += q[i] * q[i];
    return alpha / sqrt(ORC_PI) * s;
}

/* Slater correction factors of the real-space pair energy and force, Eq. 57-58
 * with beta r* = d/lambda; lambda = 0: point charges, both 1.      */
double orc_slater_BU(double d, double lambda)
{
    if (lambda <= 0.0) return 1.0;
    double x = d / lambda;
    return 1.0 - (1.0 + x) * exp(-2.0 * x);
}

double orc_slater_BF(double d, double lambda)
{
    if (lambda <= 0.0) return 1.0;
    double x = d / lambda;
    return 1.0 - (1.0 + 2.0 * x * (1.0 + x)) * exp(-2.0 * x);
}

/* Real-space (short-range) Ewald part on a sample of particles (all if ns == 0):
 *   e_i = 1/2 q_i sum'_{j,n} q_j B_U(d) erfc(alpha d)/d                 (Eq. 16-17)
 *   F_i = q_i sum'_{j,n} q_j B_F(d) [erfc(alpha d)/d^2 + (2 alpha/sqrt(pi)) exp(-alpha^2 d^2)/d] dvec/d
 * with dvec = r_i - r_j - nL, d = |dvec| <= r_cut, images |n_t| <= shells, the prime dropping
 * i = j in the home cell.  Eq. 29 prints the bracket without q_i, the unit
 * vector and the 1/d of the Gaussian term (reading R24: the bracket above is -d/dd of
 * erfc(alpha d)/d; pinned by finite differences of orc_real_energy).  B_U, B_F scale the
 * real-space energy and force terms as the paper states ("B_U and B_F are only applied on
 * real space summations"); lambda = 0 switches them off.
 * Sum_i e_i over all particles is the real-space energy.  F is ns x 3 (or N x 3).      */
void orc_real_forces(int64_t N, const double *r, const double *q, double L, double alpha,
                     double r_cut, int shells, double lambda, int64_t ns, const int64_t *sample,
                     double *F, double *e)
{
    const int64_t cnt = ns ? ns : N;
    const double two_a_sqrtpi = 2.0 * alpha / sqrt(ORC_PI);
#pragma omp parallel for schedule(dynamic, 16)
    for (int64_t t = 0; t < cnt; ++t) {
        const int64_t i = ns ? sample[t] : t;
        double fx = 0.0, fy = 0.0, fz = 0.0, ei = 0.0;
        for (int64_t j = 0; j < N; ++j)
            for (int a = -shells; a <= shells; ++a)
                for (int b = -shells; b <= shells; ++b)
                    for (int c = -shells; c <= shells; ++c) {
                        if (i == j && a == 0 && b == 0 && c == 0) continue;
                        double dx = r[3 * i] - r[3 * j] - a * L;
                        double dy = r[3 * i + 1] - r[3 * j + 1] - b * L;
                        double dz = r[3 * i + 2] - r[3 * j + 2] - c * L;
                        double d2 = dx * dx + dy * dy + dz * dz;
                        if (d2 > r_cut * r_cut) continue;
                        double d = sqrt(d2);
                        double ec = erfc(alpha * d);
                        ei += q[j] * orc_slater_BU(d, lambda) * ec / d;
                        double g = orc_slater_BF(d, lambda)
                                   * (ec / d2 + two_a_sqrtpi * exp(-alpha * alpha * d2) / d) / d;
                        fx += q[j] * g * dx; fy += q[j] * g * dy; fz += q[j] * g * dz;
                    }
        if (F) { F[3 * t] = q[i] * fx; F[3 * t + 1] = q[i] * fy; F[3 * t + 2] = q[i] * fz; }
        if (e) e[t] = 0.5 * q[i] * ei;
    }
}

/* ------------------------------------------------------------------ Oracle B */

static int wrap_index(int l, int n)
{
    int w = l % n;
    return w < 0 ? w + n : w;
}

/* Step 1 (R8-R10): u = n (x - floor x), c = floor(u + 1/2), stencil l = c-m..c+m,
 * d = u - l.  wt[t][k] = phi(d) for dimension t and stencil point k; dwt likewise phi'. */
static void stencil_weights(const double *rj, double L, int n, int m, int window, double sigma,
                            int *c, double *wt, double *dwt)
{
    for (int t = 0; t < 3; ++t) {
        double u = n * frac_pos(rj[t], L);
        c[t] = (int)floor(u + 0.5);
        for (int k = 0; k <= 2 * m; ++k) {
            double d = u - (double)(c[t] - m + k);
            wt[t * (2 * m + 1) + k] = orc_phi(window, m, sigma, d);
            if (dwt) dwt[t * (2 * m + 1) + k] = orc_dphi(window, m, sigma, d);
        }
    }
}

/* Step 3 -- spreading: g[l] += q_j phi(dx) phi(dy) phi(dz) over the
 * (2m+1)^3 stencil, naive triple loop, periodic.  g (n^3) is accumulated into.      */
void orc_spread(int64_t N, const double *r, const double *q, double L, int n, int m,
                int window, double sigma, double *g)
{
    int W = 2 * m + 1;
    double wt[3 * 64];
    int c[3];
    for (int64_t j = 0; j < N; ++j) {
        if (q[j] == 0.0) continue;
        stencil_weights(&r[3 * j], L, n, m, window, sigma, c, wt, NULL);
        for (int kz = 0; kz < W; ++kz) {
            int lz = wrap_index(c[2] - m + kz, n);
            for (int ky = 0; ky < W; ++ky) {
                int ly = wrap_index(c[1] - m + ky, n);
                double wyz = q[j] * wt[2 * W + kz] * wt[W + ky];
                for (int kx = 0; kx < W; ++kx) {
                    int lx = wrap_index(c[0] - m + kx, n);
                    g[((size_t)lz * n + ly) * n + lx] += wyz * wt[kx];
                }
            }
        }
    }
}

/* One line, plain O(n^2) DFT: out[k] = sum_l in[l] exp(sign 2 pi i k l / n), with a
 * twiddle table tw[t] = exp(sign 2 pi i t / n) indexed by (k l) mod n (R11).       */
static void dft_line(int n, int sign, const double *in_re, const double *in_im,
                     double *out_re, double *out_im)
{
    double *tr = (double *)malloc(sizeof(double) * 2 * (size_t)n), *ti = tr + n;
    for (int t = 0; t < n; ++t) {
        tr[t] = cos(2.0 * ORC_PI * t / n);
        ti[t] = sign * sin(2.0 * ORC_PI * t / n);
    }
    for (int k = 0; k < n; ++k) {
        double sr = 0.0, si = 0.0;
        for (int l = 0; l < n; ++l) {
            int t = (int)(((int64_t)k * l) % n);
            sr += in_re[l] * tr[t] - in_im[l] * ti[t];
            si += in_re[l] * ti[t] + in_im[l] * tr[t];
        }
        out_re[k] = sr;
        out_im[k] = si;
    }
    free(tr);
}

/* One line, textbook iterative radix-2 decimation-in-time FFT (n a power of two). */
static void fft_line(int n, int sign, double *re, double *im)
{
    for (int i = 1, j = 0; i < n; ++i) {            /* bit reversal */
        int bit = n >> 1;
        for (; j & bit; bit >>= 1) j ^= bit;
        j ^= bit;
        if (i < j) {
            double t = re[i]; re[i] = re[j]; re[j] = t;
            t = im[i]; im[i] = im[j]; im[j] = t;
        }
    }
    for (int len = 2; len <= n; len <<= 1) {
        for (int k = 0; k < len / 2; ++k) {
            double ang = sign * 2.0 * ORC_PI * k / len;
            double wr = cos(ang), wi = sin(ang);
            for (int i = 0; i < n; i += len) {
                int a = i + k, b = i + k + len / 2;
                double xr = re[b] * wr - im[b] * wi, xi = re[b] * wi + im[b] * wr;
                re[b] = re[a] - xr; im[b] = im[a] - xi;
                re[a] += xr; im[a] += xi;
            }
        }
    }
}

void orc_fft_line(int n, int sign, int use_dft, double *re, double *im)
{
    if (use_dft) {
        double *o = (double *)malloc(sizeof(double) * 2 * (size_t)n);
        dft_line(n, sign, re, im, o, o + n);
        memcpy(re, o, sizeof(double) * n);
        memcpy(im, o + n, sizeof(double) * n);
        free(o);
    } else {
        fft_line(n, sign, re, im);
    }
}

/* Step 4 -- unnormalised 3D transform, sign = -1 forward, +1 inverse (R11): lines
 * along x, then y, then z, each copied into a contiguous buffer.                    */
void orc_fft3d(int n, int sign, int use_dft, double *re, double *im)
{
    for (int axis = 0; axis < 3; ++axis) {
        size_t stride = axis == 0 ? 1 : (axis == 1 ? (size_t)n : (size_t)n * n);
#pragma omp parallel
        {
            double *br = (double *)malloc(sizeof(double) * 2 * (size_t)n), *bi = br + n;
#pragma omp for schedule(static)
            for (int64_t line = 0; line < (int64_t)n * n; ++line) {
                int a = (int)(line / n), b = (int)(line % n);
                size_t base = axis == 0 ? ((size_t)a * n + b) * n
                            : axis == 1 ? (size_t)a * n * n + b
                                        : (size_t)a * n + b;
                for (int l = 0; l < n; ++l) { br[l] = re[base + l * stride]; bi[l] = im[base + l * stride]; }
                orc_fft_line(n, sign, use_dft, br, bi);
                for (int l = 0; l < n; ++l) { re[base + l * stride] = br[l]; im[base + l * stride] = bi[l]; }
            }
            free(br);
        }
    }
}

static int freq_index(int k, int n) { return k < 0 ? k + n : k; }

/* Step 5 -- scaling: for n in K, S~(n) = g^[n]/D, D = Phi(nx)Phi(ny)Phi(nz);
 * E~ = (1/(2 pi L)) sum_K f^2 w |S~|^2 (Eq. 38).
 * Step 6/7 -- subdividing: writes the field spectrum on the n^3 grid,
 * zero outside K:
 *   component < 0  : psi^ = f^2 w S~/D                       (analytic variant)
 *   component 0..2 : b^_d = -i n_d f^2 w S~/D                (ik variant, Eq. 41-42)
 * gh_* is the forward transform of the spread grid; out_* may alias nothing.
 * If S_out_* != NULL (size orc_modes(k_cut)) S~ is stored in orc_modes order.     */
double orc_scale(int n, int k_cut, double L, double alpha, double lambda, int window, int m,
                 double sigma, const double *gh_re, const double *gh_im, int component,
                 double *out_re, double *out_im, double *S_out_re, double *S_out_im)
{
    size_t n3 = (size_t)n * n * n;
    if (out_re) { memset(out_re, 0, sizeof(double) * n3); memset(out_im, 0, sizeof(double) * n3); }
    double e = 0.0;
    int64_t c = 0;
    for (int nz = -k_cut; nz <= k_cut; ++nz)
        for (int ny = -k_cut; ny <= k_cut; ++ny)
            for (int nx = -k_cut; nx <= k_cut; ++nx) {
                int n2 = nx * nx + ny * ny + nz * nz;
                if (n2 == 0 || n2 > k_cut * k_cut) continue;
                size_t idx = ((size_t)freq_index(nz, n) * n + freq_index(ny, n)) * n + freq_index(nx, n);
                double D = orc_Phi(window, m, sigma, n, nx) * orc_Phi(window, m, sigma, n, ny)
                         * orc_Phi(window, m, sigma, n, nz);
                double sr = gh_re[idx] / D, si = gh_im[idx] / D;
                double fw = orc_slater_f2(n2, lambda, L) * orc_w(n2, alpha, L);
                e += fw * (sr * sr + si * si);
                if (S_out_re) { S_out_re[c] = sr; S_out_im[c] = si; }
                if (out_re) {
                    double pr = fw * sr / D, pi = fw * si / D;
                    if (component < 0) {
                        out_re[idx] = pr; out_im[idx] = pi;
                    } else {
                        int nd = component == 0 ? nx : (component == 1 ? ny : nz);
                        /* -i n_d (pr + i pi) = n_d pi - i n_d pr */
                        out_re[idx] = nd * pi; out_im[idx] = -nd * pr;
                    }
                }
                ++c;
            }
    return e / (2.0 * ORC_PI * L);
}

/* Step 6/7 -- interpolating.  field = real part of the inverse FFT.
 *   ik (component d = 0..2):  F[.,d] = (2 q_i/L^2) sum_stencil B_d[l] phi phi phi  (Eq. 42)
 *   analytic (component < 0): F[.,x] = -(q_i n/(pi L^2)) sum Psi[l] phi'(dx) phi(dy) phi(dz),
 *                             cyclic for y, z (exact gradient of E~ of step 5).
 * Forces are written (not accumulated) for the components the call covers.         */
void orc_gather(int64_t N, const double *r, const double *q, double L, int n, int m, int window,
                double sigma, int component, const double *field, double *F,
                int64_t nsample, const int64_t *sample)
{
    int W = 2 * m + 1;
    int64_t nf = nsample > 0 ? nsample : N;
#pragma omp parallel for schedule(static)
    for (int64_t s = 0; s < nf; ++s) {
        int64_t j = nsample > 0 ? sample[s] : s;
        double wt[3 * 64], dwt[3 * 64];
        int c[3];
        stencil_weights(&r[3 * j], L, n, m, window, sigma, c, wt, dwt);
        double a0 = 0.0, a1 = 0.0, a2 = 0.0;
        for (int kz = 0; kz < W; ++kz) {
            int lz = wrap_index(c[2] - m + kz, n);
            for (int ky = 0; ky < W; ++ky) {
                int ly = wrap_index(c[1] - m + ky, n);
                for (int kx = 0; kx < W; ++kx) {
                    int lx = wrap_index(c[0] - m + kx, n);
                    double v = field[((size_t)lz * n + ly) * n + lx];
                    if (component < 0) {
                        a0 += v * dwt[kx] * wt[W + ky] * wt[2 * W + kz];
                        a1 += v * wt[kx] * dwt[W + ky] * wt[2 * W + kz];
                        a2 += v * wt[kx] * wt[W + ky] * dwt[2 * W + kz];
                    } else {
                        a0 += v * wt[kx] * wt[W + ky] * wt[2 * W + kz];
                    }
                }
            }
        }
        if (component < 0) {
            double pre = -q[j] * n / (ORC_PI * L * L);
            F[3 * s] = pre * a0; F[3 * s + 1] = pre * a1; F[3 * s + 2] = pre * a2;
        } else {
            F[3 * s + component] = 2.0 * q[j] / (L * L) * a0;
        }
    }
}

/* Whole Oracle B.  variant: ORC_FORCE_ANALYTIC or ORC_FORCE_IK.  F may be NULL (energy
 * only).  grid_out (n^3) receives the spread grid if != NULL; S_out_* receive S~ in
 * orc_modes order if != NULL.  Returns 0, -1 on allocation failure, -2 on bad arguments. */
int orc_enuf(int64_t N, const double *r, const double *q, double L, double alpha, int k_cut,
             int n, int m, int window, double sigma, int variant, double lambda, int use_dft,
             double *E, double *F, int64_t nsample, const int64_t *sample,
             double *grid_out, double *S_out_re, double *S_out_im)
{
    /* the radix-2 line transform needs a power of two; the plain DFT (use_dft) is the definition for any n */
    if (n < 2 * m + 1 || ((n & (n - 1)) && !use_dft) || k_cut < 1 || 2 * k_cut > n || m < 1 || m > 20) return -2;
    size_t n3 = (size_t)n * n * n;
    double *g_re = (double *)calloc(n3, sizeof(double));
    double *g_im = (double *)calloc(n3, sizeof(double));
    double *p_re = (double *)malloc(sizeof(double) * n3);
    double *p_im = (double *)malloc(sizeof(double) * n3);
    if (!g_re || !g_im || !p_re || !p_im) { free(g_re); free(g_im); free(p_re); free(p_im); return -1; }

    orc_spread(N, r, q, L, n, m, window, sigma, g_re);
    if (grid_out) memcpy(grid_out, g_re, sizeof(double) * n3);
    orc_fft3d(n, -1, use_dft, g_re, g_im);

    if (variant == ORC_FORCE_ANALYTIC) {
        *E = orc_scale(n, k_cut, L, alpha, lambda, window, m, sigma, g_re, g_im, -1,
                       F ? p_re : NULL, p_im, S_out_re, S_out_im);
        if (F) {
            orc_fft3d(n, +1, use_dft, p_re, p_im);
            orc_gather(N, r, q, L, n, m, window, sigma, -1, p_re, F, nsample, sample);
        }
    } else {
        *E = orc_scale(n, k_cut, L, alpha, lambda, window, m, sigma, g_re, g_im, 0,
                       NULL, NULL, S_out_re, S_out_im);
        for (int d = 0; F && d < 3; ++d) {
            orc_scale(n, k_cut, L, alpha, lambda, window, m, sigma, g_re, g_im, d,
                      p_re, p_im, NULL, NULL);
            orc_fft3d(n, +1, use_dft, p_re, p_im);
            orc_gather(N, r, q, L, n, m, window, sigma, d, p_re, F, nsample, sample);
        }
    }
    free(g_re); free(g_im); free(p_re); free(p_im);
    return 0;
}

/* =================================================================== orthorhombic boxes
 * SURVEY.md section 8(f).4.  The paper treats the cubic box only and names non-cubic
 * boxes as motivation (:35, :609); this is the textbook Ewald sum of a cell with edges
 * Lb = (Lx, Ly, Lz), volume V = Lx Ly Lz, written out the same way (reading R26):
 *   x_d = r_d / L_d,  wave vector k = 2 pi h,  h = (nx/Lx, ny/Ly, nz/Lz),  n integer,
 *   S(n)  = sum_j q_j exp(-2 pi i n.x_j)                                         (Eq. 37)
 *   E_rec = (1/(2 pi V)) sum_K f^2(h) exp(-pi^2 |h|^2/alpha^2)/|h|^2 |S(n)|^2    (Eq. 38 with n/L -> h)
 *   F_i,d = (2 q_i/V) sum_K h_d f^2 exp(..)/|h|^2 Im{S e^{+2 pi i n.x_i}}        (Eq. 41 likewise)
 *   K     = { n != 0 : |h| Lmax <= k_cut },  Lmax = max(Lx, Ly, Lz)              (R26: a sphere of wave
 *           vectors; every |n_d| <= k_cut L_d/Lmax <= k_cut; the cubic K of R4 when the edges are equal)
 * With Lx = Ly = Lz all of this is the cubic case above term by term.  The ENUF steps keep ONE grid size n
 * in all three directions (grid spacing L_d/n differs per direction); only u_d = n x_d, the weights and the
 * prefactors change:  E~ = (1/(2 pi V)) sum_K f^2 w |S~|^2,
 *   analytic forces F_i,d = -(q_i n/(pi V L_d)) sum_stencil Psi[l] phi'(d_d) phi phi,
 *   ik forces       b^_d = -i h_d f^2 w S~/D,  F_i,d = (2 q_i/V) sum_stencil B_d[l] phi phi phi.
 * Pins (tests/test_oracle_pins.py): equal edges reproduce the cubic functions; a cubic system repeated
 * along one axis (box 2L x L x L, k_cut doubled) has exactly twice the energy and the same forces; forces
 * are -dE/dr by central differences per direction; Oracle B against Oracle A within the NFFT error.    */

static double box_lmax(const double *Lb)
{
    double a = Lb[0] > Lb[1] ? Lb[0] : Lb[1];
    return a > Lb[2] ? a : Lb[2];
}

/* |h|^2 Lmax^2 = nx^2 (Lmax/Lx)^2 + ny^2 (Lmax/Ly)^2 + nz^2 (Lmax/Lz)^2, in this order, fp64
 * (the membership n in K is decided on this number: <= k_cut^2)                              */
double orc_box_s(const double *Lb, int nx, int ny, int nz)
{
    double lm = box_lmax(Lb);
    double ax = (lm / Lb[0]) * (lm / Lb[0]), ay = (lm / Lb[1]) * (lm / Lb[1]), az = (lm / Lb[2]) * (lm / Lb[2]);
    return ((double)(nx * nx) * ax + (double)(ny * ny) * ay) + (double)(nz * nz) * az;
}

/* f^2(h) exp(-pi^2 |h|^2/alpha^2)/|h|^2 with |h|^2 = s/Lmax^2;  f = (1 + k^2 lambda^2/4)^-2, k = 2 pi |h| (Eq. 51, R19) */
double orc_box_fw(const double *Lb, double s, double alpha, double lambda)
{
    double lm = box_lmax(Lb);
    double h2 = s / (lm * lm);
    double w = exp(-ORC_PI * ORC_PI * h2 / (alpha * alpha)) / h2;
    if (lambda != 0.0) {
        double g = 1.0 + ORC_PI * ORC_PI * lambda * lambda * h2;
        w /= g * g * g * g;
    }
    return w;
}

int64_t orc_modes_box(int k_cut, const double *Lb, int *modes)
{
    int64_t c = 0;
    for (int nz = -k_cut; nz <= k_cut; ++nz)
        for (int ny = -k_cut; ny <= k_cut; ++ny)
            for (int nx = -k_cut; nx <= k_cut; ++nx) {
                if (nx == 0 && ny == 0 && nz == 0) continue;
                if (orc_box_s(Lb, nx, ny, nz) > (double)(k_cut * k_cut)) continue;
                if (modes) { modes[3 * c] = nx; modes[3 * c + 1] = ny; modes[3 * c + 2] = nz; }
                ++c;
            }
    return c;
}

/* Oracle A for a box.  Same contract as orc_direct. */
int orc_direct_box(int64_t N, const double *r, const double *q, const double *Lb, double alpha,
                   int k_cut, double lambda, double *E, double *F,
                   int64_t nsample, const int64_t *sample)
{
    int64_t nK = orc_modes_box(k_cut, Lb, NULL);
    int *modes = (int *)malloc(sizeof(int) * 3 * (size_t)(nK > 0 ? nK : 1));
    double *Sr = (double *)malloc(sizeof(double) * (size_t)(nK > 0 ? nK : 1));
    double *Si = (double *)malloc(sizeof(double) * (size_t)(nK > 0 ? nK : 1));
    double *x = (double *)malloc(sizeof(double) * 3 * (size_t)(N > 0 ? N : 1));
    if (!modes || !Sr || !Si || !x) { free(modes); free(Sr); free(Si); free(x); return -1; }
    orc_modes_box(k_cut, Lb, modes);
    for (int64_t j = 0; j < N; ++j)
        for (int d = 0; d < 3; ++d) x[3 * j + d] = frac_pos(r[3 * j + d], Lb[d]);
    double V = Lb[0] * Lb[1] * Lb[2];
#pragma omp parallel for schedule(static)
    for (int64_t t = 0; t < nK; ++t) {
        double sr = 0.0, si = 0.0;
        int nx = modes[3 * t], ny = modes[3 * t + 1], nz = modes[3 * t + 2];
        for (int64_t j = 0; j < N; ++j) {
            double ph = 2.0 * ORC_PI * (nx * x[3 * j] + ny * x[3 * j + 1] + nz * x[3 * j + 2]);
            sr += q[j] * cos(ph);
            si -= q[j] * sin(ph);
        }
        Sr[t] = sr; Si[t] = si;
    }
    double e = 0.0;
    for (int64_t t = 0; t < nK; ++t) {
        double s = orc_box_s(Lb, modes[3 * t], modes[3 * t + 1], modes[3 * t + 2]);
        e += orc_box_fw(Lb, s, alpha, lambda) * (Sr[t] * Sr[t] + Si[t] * Si[t]);
    }
    *E = e / (2.0 * ORC_PI * V);
    if (F) {
        int64_t nf = nsample > 0 ? nsample : N;
#pragma omp parallel for schedule(static)
        for (int64_t sI = 0; sI < nf; ++sI) {
            int64_t i = nsample > 0 ? sample[sI] : sI;
            double fx = 0.0, fy = 0.0, fz = 0.0;
            for (int64_t t = 0; t < nK; ++t) {
                int nx = modes[3 * t], ny = modes[3 * t + 1], nz = modes[3 * t + 2];
                double ph = 2.0 * ORC_PI * (nx * x[3 * i] + ny * x[3 * i + 1] + nz * x[3 * i + 2]);
                double im = Sr[t] * sin(ph) + Si[t] * cos(ph);
                double c = orc_box_fw(Lb, orc_box_s(Lb, nx, ny, nz), alpha, lambda) * im;
                fx += (nx / Lb[0]) * c; fy += (ny / Lb[1]) * c; fz += (nz / Lb[2]) * c;
            }
            double pre = 2.0 * q[i] / V;
            F[3 * sI] = pre * fx; F[3 * sI + 1] = pre * fy; F[3 * sI + 2] = pre * fz;
        }
    }
    free(modes); free(Sr); free(Si); free(x);
    return 0;
}

/* Step 1 with one edge per direction: u_d = n frac(r_d/L_d). */
static void stencil_weights_box(const double *rj, const double *Lb, int n, int m, int window, double sigma,
                                int *c, double *wt, double *dwt)
{
    for (int t = 0; t < 3; ++t) {
        double u = n * frac_pos(rj[t], Lb[t]);
        c[t] = (int)floor(u + 0.5);
        for (int k = 0; k <= 2 * m; ++k) {
            double d = u - (double)(c[t] - m + k);
            wt[t * (2 * m + 1) + k] = orc_phi(window, m, sigma, d);
            if (dwt) dwt[t * (2 * m + 1) + k] = orc_dphi(window, m, sigma, d);
        }
    }
}

/* Step 3 for a box (same triple loop as orc_spread). */
void orc_spread_box(int64_t N, const double *r, const double *q, const double *Lb, int n, int m,
                    int window, double sigma, double *g)
{
    int W = 2 * m + 1;
    double wt[3 * 64];
    int c[3];
    for (int64_t j = 0; j < N; ++j) {
        if (q[j] == 0.0) continue;
        stencil_weights_box(&r[3 * j], Lb, n, m, window, sigma, c, wt, NULL);
        for (int kz = 0; kz < W; ++kz) {
            int lz = wrap_index(c[2] - m + kz, n);
            for (int ky = 0; ky < W; ++ky) {
                int ly = wrap_index(c[1] - m + ky, n);
                double wyz = q[j] * wt[2 * W + kz] * wt[W + ky];
                for (int kx = 0; kx < W; ++kx) {
                    int lx = wrap_index(c[0] - m + kx, n);
                    g[((size_t)lz * n + ly) * n + lx] += wyz * wt[kx];
                }
            }
        }
    }
}

/* Step 5 and the subdividing of step 6/7 for a box; same contract as orc_scale, S~ in orc_modes_box order. */
double orc_scale_box(int n, int k_cut, const double *Lb, double alpha, double lambda, int window, int m,
                     double sigma, const double *gh_re, const double *gh_im, int component,
                     double *out_re, double *out_im, double *S_out_re, double *S_out_im)
{
    size_t n3 = (size_t)n * n * n;
    if (out_re) { memset(out_re, 0, sizeof(double) * n3); memset(out_im, 0, sizeof(double) * n3); }
    double e = 0.0;
    int64_t c = 0;
    for (int nz = -k_cut; nz <= k_cut; ++nz)
        for (int ny = -k_cut; ny <= k_cut; ++ny)
            for (int nx = -k_cut; nx <= k_cut; ++nx) {
                if (nx == 0 && ny == 0 && nz == 0) continue;
                double s = orc_box_s(Lb, nx, ny, nz);
                if (s > (double)(k_cut * k_cut)) continue;
                size_t idx = ((size_t)freq_index(nz, n) * n + freq_index(ny, n)) * n + freq_index(nx, n);
                double D = orc_Phi(window, m, sigma, n, nx) * orc_Phi(window, m, sigma, n, ny)
                         * orc_Phi(window, m, sigma, n, nz);
                double sr = gh_re[idx] / D, si = gh_im[idx] / D;
                double fw = orc_box_fw(Lb, s, alpha, lambda);
                e += fw * (sr * sr + si * si);
                if (S_out_re) { S_out_re[c] = sr; S_out_im[c] = si; }
                if (out_re) {
                    double pr = fw * sr / D, pi = fw * si / D;
                    if (component < 0) {
                        out_re[idx] = pr; out_im[idx] = pi;
                    } else {
                        double hd = component == 0 ? nx / Lb[0] : (component == 1 ? ny / Lb[1] : nz / Lb[2]);
                        out_re[idx] = hd * pi; out_im[idx] = -hd * pr;      /* -i h_d (pr + i pi) */
                    }
                }
                ++c;
            }
    return e / (2.0 * ORC_PI * Lb[0] * Lb[1] * Lb[2]);
}

/* Step 6/7 interpolation for a box; same contract as orc_gather. */
void orc_gather_box(int64_t N, const double *r, const double *q, const double *Lb, int n, int m, int window,
                    double sigma, int component, const double *field, double *F,
                    int64_t nsample, const int64_t *sample)
{
    int W = 2 * m + 1;
    int64_t nf = nsample > 0 ? nsample : N;
    double V = Lb[0] * Lb[1] * Lb[2];
#pragma omp parallel for schedule(static)
    for (int64_t s = 0; s < nf; ++s) {
        int64_t j = nsample > 0 ? sample[s] : s;
        double wt[3 * 64], dwt[3 * 64];
        int c[3];
        stencil_weights_box(&r[3 * j], Lb, n, m, window, sigma, c, wt, dwt);
        double a0 = 0.0, a1 = 0.0, a2 = 0.0;
        for (int kz = 0; kz < W; ++kz) {
            int lz = wrap_index(c[2] - m + kz, n);
            for (int ky = 0; ky < W; ++ky) {
                int ly = wrap_index(c[1] - m + ky, n);
                for (int kx = 0; kx < W; ++kx) {
                    int lx = wrap_index(c[0] - m + kx, n);
                    double v = field[((size_t)lz * n + ly) * n + lx];
                    if (component < 0) {
                        a0 += v * dwt[kx] * wt[W + ky] * wt[2 * W + kz];
                        a1 += v * wt[kx] * dwt[W + ky] * wt[2 * W + kz];
                        a2 += v * wt[kx] * wt[W + ky] * dwt[2 * W + kz];
                    } else {
                        a0 += v * wt[kx] * wt[W + ky] * wt[2 * W + kz];
                    }
                }
            }
        }
        if (component < 0) {
            double pre = -q[j] * n / (ORC_PI * V);
            F[3 * s] = pre / Lb[0] * a0; F[3 * s + 1] = pre / Lb[1] * a1; F[3 * s + 2] = pre / Lb[2] * a2;
        } else {
            F[3 * s + component] = 2.0 * q[j] / V * a0;
        }
    }
}

/* Whole Oracle B for a box; same contract as orc_enuf. */
int orc_enuf_box(int64_t N, const double *r, const double *q, const double *Lb, double alpha, int k_cut,
                 int n, int m, int window, double sigma, int variant, double lambda, int use_dft,
                 double *E, double *F, int64_t nsample, const int64_t *sample,
                 double *grid_out, double *S_out_re, double *S_out_im)
{
    /* the radix-2 line transform needs a power of two; the plain DFT (use_dft) is the definition for any n */
    if (n < 2 * m + 1 || ((n & (n - 1)) && !use_dft) || k_cut < 1 || 2 * k_cut > n || m < 1 || m > 20) return -2;
    size_t n3 = (size_t)n * n * n;
    double *g_re = (double *)calloc(n3, sizeof(double));
    double *g_im = (double *)calloc(n3, sizeof(double));
    double *p_re = (double *)malloc(sizeof(double) * n3);
    double *p_im = (double *)malloc(sizeof(double) * n3);
    if (!g_re || !g_im || !p_re || !p_im) { free(g_re); free(g_im); free(p_re); free(p_im); return -1; }

    orc_spread_box(N, r, q, Lb, n, m, window, sigma, g_re);
    if (grid_out) memcpy(grid_out, g_re, sizeof(double) * n3);
    orc_fft3d(n, -1, use_dft, g_re, g_im);

    if (variant == ORC_FORCE_ANALYTIC) {
        *E = orc_scale_box(n, k_cut, Lb, alpha, lambda, window, m, sigma, g_re, g_im, -1,
                           F ? p_re : NULL, p_im, S_out_re, S_out_im);
        if (F) {
            orc_fft3d(n, +1, use_dft, p_re, p_im);
            orc_gather_box(N, r, q, Lb, n, m, window, sigma, -1, p_re, F, nsample, sample);
        }
    } else {
        *E = orc_scale_box(n, k_cut, Lb, alpha, lambda, window, m, sigma, g_re, g_im, 0,
                           NULL, NULL, S_out_re, S_out_im);
        for (int d = 0; F && d < 3; ++d) {
            orc_scale_box(n, k_cut, Lb, alpha, lambda, window, m, sigma, g_re, g_im, d,
                          p_re, p_im, NULL, NULL);
            orc_fft3d(n, +1, use_dft, p_re, p_im);
            orc_gather_box(N, r, q, Lb, n, m, window, sigma, d, p_re, F, nsample, sample);
        }
    }
    free(g_re); free(g_im); free(p_re); free(p_im);
    return 0;
}
