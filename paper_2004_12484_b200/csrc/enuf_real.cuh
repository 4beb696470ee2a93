// Real-space (short-range) part of the Ewald sum, SURVEY 8(f).1 -- Eq. 16-17,
// Eq. 29 (:243, reading R24) and the self term Eq. 24 (:216):
//   E_real = 1/2 sum'_{i,j} q_i q_j B_U(d) erfc(alpha d)/d,          d = |r_i - r_j|_min-image <= r_cut
//   F_i    = q_i sum'_j q_j B_F(d) [erfc(alpha d)/d^2 + (2 alpha/sqrt(pi)) exp(-alpha^2 d^2)/d] (r_i - r_j)/d
//   E_self = (alpha/sqrt(pi)) sum_i q_i^2
// B_U, B_F are the Slater factors of Eq. 57-58 (:434-436), 1 for point charges.
//
// The paper's "Near Distance" scheme is a linked-cell list whose cells are
// smaller than the cutoff.  Here: charged particles are counting-sorted into ncd^3 cells of side
// L/ncd >= r_cut/2 (neighbour range s = 2 cells; boxes with fewer than 5 such cells per dimension use a
// single cell = all pairs), x fastest, with the scan kernels of enuf_bin.cuh; one thread per sorted particle walks
// the (2s+1)^2 rows of neighbouring cells -- the 2s+1 cells of a row are contiguous in the sorted
// array, split in two where the row wraps around the box -- and applies the minimum image.
#pragma once

#include "enuf_bin.cuh"
#include "enuf_common.cuh"

namespace enuf {

// erfc for the fp32 pair term: erfc(x) = exp(-x^2) t P(u), t = 1/(1 + x/2), u = ua t + ub in [-1, 1], with P
// the degree-10 Chebyshev interpolant (as monomials in u) of exp(x^2) erfc(x)/t on 0 <= x <= alpha r_cut,
// fitted in fp64 when the real-space part is first used (relative error <= 4e-9 for alpha r_cut <= 8, far
// below fp32 rounding).  The exponential is the one the Gaussian term of the force needs anyway, so the
// pair term costs one expf instead of erfcf + expf.
struct ErfcFit {
    float c[kErfcDeg + 1];
    float ua, ub;
};

struct RealGeom {
    int ncd;        // cells per dimension
    int s;          // neighbour range in cells (0: single cell, all pairs)
    double L;
};

__device__ __forceinline__ float r_erfc(float x) { return erfcf(x); }
__device__ __forceinline__ double r_erfc(double x) { return erfc(x); }
__device__ __forceinline__ float r_rint(float x) { return rintf(x); }
__device__ __forceinline__ double r_rint(double x) { return rint(x); }

// position wrapped into [0, L) (kept bit-exact when it already lies there) and its cell
template <typename T>
__device__ __forceinline__ void real_locate(const T* __restrict__ r, int64_t j, const RealGeom& g, T (&p)[3], int& cell) {
    int c[3];
#pragma unroll
    for (int t = 0; t < 3; ++t) {
        const double v = (double)r[3 * j + t];
        double w = v;
        if (!(v >= 0.0 && v < g.L)) {
            double x = v / g.L;
            x -= floor(x);
            w = x * g.L;
            if (w >= g.L) w = 0.0;
        }
        p[t] = (T)w;
        // the cell is taken from the STORED (rounded) coordinate, the one the distances use
        int ci = (int)((double)p[t] * ((double)g.ncd / g.L));
        c[t] = ci >= g.ncd ? g.ncd - 1 : ci;
    }
    cell = (c[2] * g.ncd + c[1]) * g.ncd + c[0];
}

template <typename T>
__global__ void __launch_bounds__(256)
real_count_kernel(const T* __restrict__ r, const T* __restrict__ q, T* __restrict__ F, int zero_neutral,
                  int64_t N, RealGeom g, uint32_t* __restrict__ count) {
    const int64_t j = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (j >= N) return;
    if (q[j] == (T)0) {
        if (zero_neutral) { F[3 * j] = (T)0; F[3 * j + 1] = (T)0; F[3 * j + 2] = (T)0; }
        return;
    }
    T p[3];
    int cell;
    real_locate(r, j, g, p, cell);
    atomicAdd(&count[cell], 1u);
}

template <typename T>
__global__ void __launch_bounds__(256)
real_scatter_kernel(const T* __restrict__ r, const T* __restrict__ q, int64_t N, RealGeom g,
                    uint32_t* __restrict__ cursor, typename Vec4<T>::type* __restrict__ pos,
                    uint32_t* __restrict__ idx) {
    const int64_t j = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (j >= N) return;
    const T qj = q[j];
    if (qj == (T)0) return;
    T p[3];
    int cell;
    real_locate(r, j, g, p, cell);
    const uint32_t slot = atomicAdd(&cursor[cell], 1u);
    typename Vec4<T>::type v;
    v.x = p[0]; v.y = p[1]; v.z = p[2]; v.w = qj;
    pos[slot] = v;
    idx[slot] = (uint32_t)j;
}

constexpr int kRealThreads = 128;

// One thread per sorted (charged) particle.  partial[2 b], partial[2 b + 1]: the CTA's sums of
// q_i sum_j q_j B_U erfc/d (twice the pair energy) and of q_i^2, in fp64.
template <typename T, bool kSlater>
__global__ void __launch_bounds__(kRealThreads)
real_force_kernel(const typename Vec4<T>::type* __restrict__ pos, const uint32_t* __restrict__ idx,
                  const uint32_t* __restrict__ offset, int ncells, RealGeom g, T alpha, T r_cut2,
                  T inv_lambda, const __grid_constant__ ErfcFit ef, int accumulate, T* __restrict__ F,
                  double* __restrict__ partial) {
    using V4 = typename Vec4<T>::type;
    const uint32_t i = blockIdx.x * kRealThreads + threadIdx.x;
    const uint32_t n_sorted = offset[ncells];          // number of charged particles
    double e_acc = 0.0, q2_acc = 0.0;
    if (i < n_sorted) {
        const V4 pi = pos[i];
        const T two_a_sqrtpi = (T)(2.0 * 0.56418958354775628694807945156077) * alpha;   // 2 alpha / sqrt(pi)
        int cx, cy, cz;
        {
            const double sc = (double)g.ncd / g.L;
            cx = min((int)((double)pi.x * sc), g.ncd - 1);
            cy = min((int)((double)pi.y * sc), g.ncd - 1);
            cz = min((int)((double)pi.z * sc), g.ncd - 1);
        }
        T fx = (T)0, fy = (T)0, fz = (T)0;
        T e_run = (T)0;
        // one pair at separation (dx, dy, dz) = r_i - r_j (image applied)
        auto pair = [&](const V4& pj, T dx, T dy, T dz, bool other) {
            const T d2 = dx * dx + dy * dy + dz * dz;
            if (d2 <= r_cut2 && other) {
                T d, inv_d;
                if (sizeof(T) == 4) {
                    // 1/d by the reciprocal-square-root unit and one Newton step (relative error ~1e-7), d = d2 / d:
                    // no IEEE square root and division (each a MUFU plus a fix-up sequence with a slow path)
                    const float d2f = (float)d2;
                    float y = rsqrtf(d2f);
                    y = y * fmaf(-0.5f * d2f, y * y, 1.5f);
                    inv_d = (T)y; d = (T)(d2f * y);
                } else {
                    d = r_sqrt(d2); inv_d = (T)1 / d;
                }
                const T ad = alpha * d;
                const T ex = r_exp(-ad * ad);
                T ec;
                if (sizeof(T) == 4) {
                    const float t = __fdividef(1.0f, fmaf(0.5f, (float)ad, 1.0f)), u = fmaf(t, ef.ua, ef.ub);
                    float P = ef.c[kErfcDeg];
#pragma unroll
                    for (int k = kErfcDeg - 1; k >= 0; --k) P = fmaf(P, u, ef.c[k]);
                    ec = (T)(t * P) * ex;
                } else {
                    ec = r_erfc(ad);
                }
                T eterm = ec * inv_d;
                T g_ = (eterm * inv_d + two_a_sqrtpi * ex * inv_d) * inv_d;
                if (kSlater) {
                    const T x = d * inv_lambda, ex = r_exp(-(T)2 * x);
                    eterm *= (T)1 - ((T)1 + x) * ex;                           // B_U, Eq. 57
                    g_ *= (T)1 - ((T)1 + (T)2 * x * ((T)1 + x)) * ex;          // B_F, Eq. 58
                }
                e_run += pj.w * eterm;
                const T qg = pj.w * g_;
                fx += qg * dx; fy += qg * dy; fz += qg * dz;
            }
        };
        if (g.s == 0) {
            // one cell: all pairs, minimum image taken in fp64 (small systems only)
            for (uint32_t j = 0; j < n_sorted; ++j) {
                const V4 pj = pos[j];
                double dx = (double)pi.x - (double)pj.x, dy = (double)pi.y - (double)pj.y, dz = (double)pi.z - (double)pj.z;
                dx -= g.L * rint(dx / g.L); dy -= g.L * rint(dy / g.L); dz -= g.L * rint(dz / g.L);
                pair(pj, (T)dx, (T)dy, (T)dz, j != i);
            }
            e_acc += (double)e_run;
        } else {
            // The image shift of a neighbouring cell is known from the cell wrap.  With stored coordinates in
            // [0, L) the separation is formed as  A - (r_j - B)  with (A, B) per segment chosen so that every
            // subtraction has a small result (no cancellation against L in fp32):
            //   no wrap            A = r_i,               B = 0
            //   j near L, i near 0 A = r_i + (L - Lhi),   B = Lhi = (T) L       [r_j - Lhi is exact]
            //   j near 0, i near L A = r_i - L (in fp64), B = 0
            const int s = g.s, ncd = g.ncd;
            const T Lhi = (T)g.L;
            const double Llo = g.L - (double)Lhi;
            auto shifted = [&](T ri, int wrap, T& A, T& B) {
                if (wrap < 0) { A = (T)((double)ri + Llo); B = Lhi; }
                else if (wrap > 0) { A = (T)((double)ri - g.L); B = (T)0; }
                else { A = ri; B = (T)0; }
            };
            auto range = [&](uint32_t j0, uint32_t j1, T Ax, T Bx, T Ay, T By, T Az, T Bz) {
                for (uint32_t j = j0; j < j1; ++j) {
                    const V4 pj = pos[j];
                    pair(pj, Ax - (pj.x - Bx), Ay - (pj.y - By), Az - (pj.z - Bz), j != i);
                }
                e_acc += (double)e_run;
                e_run = (T)0;
            };
            for (int oz = -s; oz <= s; ++oz) {
                int z = cz + oz;
                const int wz = z < 0 ? -1 : (z >= ncd ? 1 : 0);
                z -= wz * ncd;
                T Az, Bz; shifted(pi.z, wz, Az, Bz);
                for (int oy = -s; oy <= s; ++oy) {
                    int y = cy + oy;
                    const int wy = y < 0 ? -1 : (y >= ncd ? 1 : 0);
                    y -= wy * ncd;
                    T Ay, By; shifted(pi.y, wy, Ay, By);
                    const int row = (z * ncd + y) * ncd;
                    const int x0 = cx - s, x1 = cx + s;
                    // in-box part of the row, then the part that wraps (2 s + 1 <= ncd: no overlap)
                    range(offset[row + max(x0, 0)], offset[row + min(x1, ncd - 1) + 1], pi.x, (T)0, Ay, By, Az, Bz);
                    if (x0 < 0) {
                        T Ax, Bx; shifted(pi.x, -1, Ax, Bx);
                        range(offset[row + ncd + x0], offset[row + ncd], Ax, Bx, Ay, By, Az, Bz);
                    }
                    if (x1 >= ncd) {
                        T Ax, Bx; shifted(pi.x, 1, Ax, Bx);
                        range(offset[row], offset[row + x1 - ncd + 1], Ax, Bx, Ay, By, Az, Bz);
                    }
                }
            }
        }
        const size_t j = (size_t)idx[i];
        const T qi = pi.w;
        if (accumulate) {
            F[3 * j] += qi * fx; F[3 * j + 1] += qi * fy; F[3 * j + 2] += qi * fz;
        } else {
            F[3 * j] = qi * fx; F[3 * j + 1] = qi * fy; F[3 * j + 2] = qi * fz;
        }
        e_acc *= (double)qi;
        q2_acc = (double)qi * (double)qi;
    }
    // CTA sums in a fixed order
    __shared__ double red[2][kRealThreads];
    red[0][threadIdx.x] = e_acc; red[1][threadIdx.x] = q2_acc;
    __syncthreads();
    for (int o = kRealThreads / 2; o > 0; o >>= 1) {
        if ((int)threadIdx.x < o) {
            red[0][threadIdx.x] += red[0][threadIdx.x + o];
            red[1][threadIdx.x] += red[1][threadIdx.x + o];
        }
        __syncthreads();
    }
    if (threadIdx.x == 0) { partial[2 * blockIdx.x] = red[0][0]; partial[2 * blockIdx.x + 1] = red[1][0]; }
}

// e_out[0] = e_scale * sum partial[2 b], e_out[1] = self_scale * sum partial[2 b + 1]; fixed order, one CTA
static __global__ void __launch_bounds__(256)
real_energy_finish_kernel(const double* __restrict__ partial, int count, double e_scale, double self_scale,
                          double* __restrict__ e_out) {
    __shared__ double red[2][256];
    double a = 0.0, b = 0.0;
    for (int i = threadIdx.x; i < count; i += 256) { a += partial[2 * i]; b += partial[2 * i + 1]; }
    red[0][threadIdx.x] = a; red[1][threadIdx.x] = b;
    __syncthreads();
    for (int o = 128; o > 0; o >>= 1) {
        if ((int)threadIdx.x < o) { red[0][threadIdx.x] += red[0][threadIdx.x + o]; red[1][threadIdx.x] += red[1][threadIdx.x + o]; }
        __syncthreads();
    }
    if (threadIdx.x == 0) { e_out[0] = e_scale * red[0][0]; e_out[1] = self_scale * red[1][0]; }
}

}  // namespace enuf
