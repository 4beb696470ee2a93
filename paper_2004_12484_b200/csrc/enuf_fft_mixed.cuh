// Steps a3, a4, a5 for grids of n = 3 * 2^k points per dimension (48, 96, 192, 384): the oversampling factor
// sigma_s = 1.5 of the paper's parameter sweep (Fig. 1 :360) with M = 32 ... 256.  The fused,
// pruned five-pass FFT of enuf_fft.cuh is built on the 16 x n/16 shape of a power of two; these sizes take a plain
// path instead -- correct and measured, not tuned:
//   X forward  G (real) -> C (complex n^3),  Y, Z forward in place,
//   scale      S~ = g^/D, E partials (fp64), psi^ = f^2 w S~/D  (or the three b^_d of the ik variant), pointwise,
//   Z, Y inverse in place, X inverse C -> G (real part),
// every line transform a Stockham autosort FFT in shared memory (one radix-3 step, then radix-4 steps and at most one radix-2 step; the
// twiddles exp(-2 pi i j/n) come from a table made in fp64 on the host).  Same conventions as the oracle (R11:
// forward e^-, inverse e^+, both unnormalised; R4, R12 for the mode set; R26 for orthorhombic boxes).
#pragma once

#include "enuf_common.cuh"
#include "enuf_fft.cuh"      // Cx arithmetic, ScaleTables, z_pass_energy_finish

namespace enuf {

// lines per CTA: 16 (fp32: 128 contiguous bytes across the lines of a strided pass) or 8 (fp64); n^2 is a multiple of 16.
// The line pitch in shared memory is n + 1 complex values (n is a multiple of 16: without the pad the lines of a CTA
// would start in the same bank).
template <typename T> constexpr int mix_lines() { return sizeof(T) == 4 ? 16 : 8; }
template <typename T> size_t fft_mixed_smem_bytes(int n) { return 2 * sizeof(Cx<T>) * (size_t)mix_lines<T>() * (n + 1); }

// One Stockham step of radix R on the lines of a CTA (length n, kFftThreads / nl threads per line): src -> dst.
// Ns = product of the radices already done = 1 (the radix-3 step) or 3 * 2^sh (the radix-4 and radix-2 steps).
// Item j in [0, n/R): v[r] = src[j + r n/R] w^(r (j mod Ns) n/(Ns R)), DFT_R, dst[(j / Ns) Ns R + (j mod Ns) + r Ns] = v[r]
// (r (j mod Ns) n/(Ns R) < n: the table index needs no reduction; j / Ns = (j >> sh) / 3: no division by a run-time value).
template <typename T, int R>
__device__ __forceinline__ void mix_step(const Cx<T>* __restrict__ src, Cx<T>* __restrict__ dst, int n, int nl, int sh,
                                         int sign, const Cx<T>* __restrict__ tw) {
    const int per = n / R, pitch = n + 1, tpl = kFftThreads / nl;
    const int Ns = R == 3 ? 1 : 3 << sh, tstep = per / Ns;
    const int l = threadIdx.x / tpl;
    const Cx<T>* s = src + (size_t)l * pitch;
    Cx<T>* dl = dst + (size_t)l * pitch;
    for (int j = threadIdx.x - l * tpl; j < per; j += tpl) {
        const int jq = R == 3 ? j : (j >> sh) / 3, k = j - jq * Ns;
        Cx<T> v[R];
#pragma unroll
        for (int r = 0; r < R; ++r) {
            v[r] = s[j + r * per];
            if (r > 0 && k > 0) {
                Cx<T> w = __ldg(&tw[r * k * tstep]);
                if (sign > 0) w.y = -w.y;
                v[r] = cx_mul(v[r], w);
            }
        }
        Cx<T>* d = dl + jq * Ns * R + k;
        if (R == 2) {
            d[0] = cx_add(v[0], v[1]);
            d[Ns] = cx_sub(v[0], v[1]);
        } else if (R == 4) {
            // DFT_4: X1 = (a - c) + w (b - d), X3 = (a - c) - w (b - d), w = exp(sign 2 pi i/4) = sign i
            const Cx<T> s02 = cx_add(v[0], v[2]), d02 = cx_sub(v[0], v[2]), s13 = cx_add(v[1], v[3]), d13 = cx_sub(v[1], v[3]);
            const Cx<T> rot = sign < 0 ? cx_make<T>(d13.y, -d13.x) : cx_make<T>(-d13.y, d13.x);
            d[0] = cx_add(s02, s13);
            d[Ns] = cx_add(d02, rot);
            d[2 * Ns] = cx_sub(s02, s13);
            d[3 * Ns] = cx_sub(d02, rot);
        } else {
            // DFT_3: X1 = a + b w + c w^2, X2 = a + b w^2 + c w, w = exp(sign 2 pi i/3) = (-1/2, sign sqrt(3)/2)
            const T h = (T)0.86602540378443864676 * (T)(sign < 0 ? -1 : 1);
            const Cx<T> sum = cx_add(v[1], v[2]), dif = cx_sub(v[1], v[2]);
            const Cx<T> m = cx_make<T>(v[0].x - (T)0.5 * sum.x, v[0].y - (T)0.5 * sum.y);
            const Cx<T> rot = cx_make<T>(-h * dif.y, h * dif.x);          // i h (b - c)
            d[0] = cx_add(v[0], sum);
            d[Ns] = cx_add(m, rot);
            d[2 * Ns] = cx_sub(m, rot);
        }
    }
}

// Line transforms along one direction.  Line id -> first element (id / n) A + (id % n) B, element stride `stride`
// (x: A = n^2, B = n, stride 1;  y: A = n^2, B = 1, stride n;  z: A = n, B = 1, stride n^2), all in elements.
// kAlongX: the elements of a line are contiguous (loads run along the line), else the lines of a CTA are
// (consecutive x: loads run across the lines).  kRealIn / kRealOut: the X passes read / write the real grid.
template <typename T, bool kRealIn, bool kRealOut, bool kAlongX>
__global__ void __launch_bounds__(kFftThreads)
fft_mixed_kernel(const void* __restrict__ in, void* __restrict__ out, int n, size_t A, size_t B, size_t stride, int sign,
                 const Cx<T>* __restrict__ tw) {
    pdl_prologue();
    extern __shared__ __align__(16) unsigned char smem_raw[];
    constexpr int kMixLines = mix_lines<T>();
    const int pitch = n + 1;
    Cx<T>* s0 = reinterpret_cast<Cx<T>*>(smem_raw);
    Cx<T>* s1 = s0 + (size_t)kMixLines * pitch;
    // a thread stays with one line: along x the tpl threads of a line run along it, otherwise consecutive threads take
    // consecutive lines (= consecutive x) of the same element index
    constexpr int tpl = kFftThreads / kMixLines;
    const int l = kAlongX ? threadIdx.x / tpl : threadIdx.x % kMixLines;
    const int i0 = kAlongX ? threadIdx.x % tpl : threadIdx.x / kMixLines;
    const int id = blockIdx.x * kMixLines + l;
    const size_t base = (size_t)(id / n) * A + (size_t)(id % n) * B;
    for (int i = i0; i < n; i += tpl) {
        const size_t off = base + (size_t)i * stride;
        Cx<T> v;
        if (kRealIn) { v.x = static_cast<const T*>(in)[off]; v.y = (T)0; }
        else v = static_cast<const Cx<T>*>(in)[off];
        s0[(size_t)l * pitch + i] = v;
    }
    __syncthreads();
    Cx<T>* src = s0;
    Cx<T>* dst = s1;
    mix_step<T, 3>(src, dst, n, kMixLines, 0, sign, tw);
    __syncthreads();
    { Cx<T>* t = src; src = dst; dst = t; }
    int sh = 0;
    for (; (12 << sh) <= n; sh += 2) {                       // radix-4 steps while a factor 4 is left ..
        mix_step<T, 4>(src, dst, n, kMixLines, sh, sign, tw);
        __syncthreads();
        Cx<T>* t = src; src = dst; dst = t;
    }
    if ((3 << sh) < n) {                                     // .. and one radix-2 step for an odd power of two
        mix_step<T, 2>(src, dst, n, kMixLines, sh, sign, tw);
        __syncthreads();
        Cx<T>* t = src; src = dst; dst = t;
    }
    for (int i = i0; i < n; i += tpl) {
        const size_t off = base + (size_t)i * stride;
        const Cx<T> v = src[(size_t)l * pitch + i];
        if (kRealOut) static_cast<T*>(out)[off] = v.x;
        else static_cast<Cx<T>*>(out)[off] = v;
    }
}

// Scaling, energy and subdividing on the full complex spectrum C0[kz][ky][kx] (signed frequencies k = i for
// i <= n/2, i - n above): for 0 < |k|^2 <= k_cut^2 (R4, R12)
//   S~ = g^ iphi[|kx|] iphi[|ky|] iphi[|kz|],  E += wf[|k|^2] |S~|^2  (every mode of the full space once),
//   psi^ = wf S~ iphi iphi iphi  (NOUT = 1)  or  b^_d = -i n_d psi^ into C0, C1, C2  (NOUT = 3); zero elsewhere.
// The energy partials are summed by the last CTA in a fixed order (z_pass_energy_finish).
// kBox (orthorhombic plans, R26): membership and weight from s = |h|^2 Lmax^2 formed in fp64 in the same order
// as the fused Z pass (fft_z_fused_kernel), b^_d = -i h_d psi^ with h_d = n_d / L_d.
template <typename T, int NOUT, bool kBox = false>
__global__ void __launch_bounds__(kFftThreads)
mixed_scale_kernel(Cx<T>* __restrict__ C0, Cx<T>* __restrict__ C1, Cx<T>* __restrict__ C2, int n, int kcut, int Kxp, int Ky,
                   ScaleTables st, double* __restrict__ e_partial, Cx<T>* __restrict__ spectrum,
                   unsigned* __restrict__ done_count, double e_scale, double* __restrict__ e_out, const BoxScale bs) {
    pdl_prologue();
    __shared__ double red[kFftThreads / 32];
    const T* iphi = static_cast<const T*>(st.iphi);
    const T* wf = static_cast<const T*>(st.wf);
    const size_t n3 = (size_t)n * n * n;
    const int kc2 = kcut * kcut;
    double e_acc = 0.0;
    for (size_t idx = (size_t)blockIdx.x * kFftThreads + threadIdx.x; idx < n3; idx += (size_t)gridDim.x * kFftThreads) {
        const int ix = (int)(idx % n), iy = (int)((idx / n) % n), iz = (int)(idx / ((size_t)n * n));
        const int kx = ix <= n / 2 ? ix : ix - n, ky = iy <= n / 2 ? iy : iy - n, kz = iz <= n / 2 ? iz : iz - n;
        const int ax = kx < 0 ? -kx : kx, ay = ky < 0 ? -ky : ky, az = kz < 0 ? -kz : kz;
        const int s = kx * kx + ky * ky + kz * kz;
        Cx<T> o = cx_make<T>((T)0, (T)0);
        bool in_k = ax <= kcut && ay <= kcut && az <= kcut && s > 0;
        T w = (T)0;
        if constexpr (kBox) {
            const double sxy = __dadd_rn(__dmul_rn((double)(kx * kx), bs.a[0]), __dmul_rn((double)(ky * ky), bs.a[1]));
            const double sb = __dadd_rn(sxy, __dmul_rn((double)(kz * kz), bs.a[2]));
            in_k = in_k && sxy <= (double)kc2 && sb <= (double)kc2;
            if (in_k) {
                constexpr double PI = 3.14159265358979323846264338327950288;
                const double h2 = sb / bs.lm2;
                double wd = exp(-PI * PI * h2 / (bs.alpha * bs.alpha)) / h2;
                if (bs.lambda != 0.0) {
                    const double gq = 1.0 + PI * PI * bs.lambda * bs.lambda * h2;
                    wd /= (gq * gq) * (gq * gq);
                }
                w = (T)wd;
            }
        } else {
            in_k = in_k && s <= kc2;
            if (in_k) w = wf[s];
        }
        if (in_k) {
            const T ip3 = iphi[ax] * iphi[ay] * iphi[az];
            const Cx<T> g = C0[idx];
            const Cx<T> S = cx_make<T>(g.x * ip3, g.y * ip3);
            e_acc += (double)w * ((double)S.x * (double)S.x + (double)S.y * (double)S.y);
            if (spectrum && kx >= 0) {
                const int kyp = ky >= 0 ? ky : ky + Ky, kzp = kz >= 0 ? kz : kz + Ky;
                spectrum[((size_t)kzp * Ky + kyp) * Kxp + kx] = S;
            }
            const T sc = w * ip3;
            o = cx_make<T>(S.x * sc, S.y * sc);
        }
        if (NOUT == 1) {
            C0[idx] = o;
        } else {
            // b^_d = -i n_d psi^ :  -i (x + i y) = y - i x
            const T hx = kBox ? (T)((double)kx / bs.l[0]) : (T)kx, hy = kBox ? (T)((double)ky / bs.l[1]) : (T)ky,
                    hz = kBox ? (T)((double)kz / bs.l[2]) : (T)kz;
            C0[idx] = cx_make<T>(hx * o.y, -hx * o.x);
            C1[idx] = cx_make<T>(hy * o.y, -hy * o.x);
            C2[idx] = cx_make<T>(hz * o.y, -hz * o.x);
        }
    }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) e_acc += __shfl_xor_sync(0xffffffffu, e_acc, o);
    if ((threadIdx.x & 31) == 0) red[threadIdx.x >> 5] = e_acc;
    __syncthreads();
    double sum = 0.0;
    if (threadIdx.x == 0) {
#pragma unroll
        for (int w = 0; w < kFftThreads / 32; ++w) sum += red[w];
    }
    z_pass_energy_finish(sum, e_partial, done_count, e_scale, e_out);
}

}  // namespace enuf
