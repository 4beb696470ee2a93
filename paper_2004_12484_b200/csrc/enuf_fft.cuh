// Steps a3, a4, a5 -- uniform 3D FFT of the oversampled grid, with
// the scaling / subdividing steps and the energy sum fused into the z pass.  Hand-written
// shared-memory FFT, n in {32, 64, 128, 256}; no cuFFT in the product path.
//
// One line of length N is transformed by TPL = N/16 threads in two register passes with
// one shared-memory exchange (four-step FFT, N = RA*RB):
//   pass A: for each a in [0,RB):  DFT_RA over n1 of x[RB*n1 + a], times W_N^(a*k1)
//   pass B: for each k1 in [0,RA): DFT_RB over a            ->  X[k1 + RA*k2]
// forward uses (RA, RB) = (16, N/16), inverse (N/16, 16), so the registers a thread holds
// after a forward pass B are exactly its inputs of an inverse pass A: the fused z pass goes
// forward -> scale -> inverse without touching memory in between.
//
// Data layout (x fastest everywhere), pruned to the modes the Ewald sphere can reach:
//   G  [z][y][x]        real      n^3
//   A1 [z][y][kx]       complex   kx in [0, Kxp), Kxp = roundup(k_cut+1, 8); kx > k_cut are 0
//   A2 [z][ky'][kx]     complex   ky' in [0, Ky), Ky = 2 k_cut+1; ky' <= k_cut is ky = ky',
//                                 ky' > k_cut is ky = ky' - Ky (negative frequencies)
// Passes: X fwd G->A1, Y fwd A1->A2, Z fused A2->A2 (in place), Y inv A2->A1, X inv A1->G.
#pragma once

#include "enuf_common.cuh"

namespace enuf {

template <typename T> __device__ __forceinline__ Cx<T> cx_make(T a, T b) { Cx<T> r; r.x = a; r.y = b; return r; }
// Complex arithmetic.  fp32 uses the packed two-lane instructions of sm_100a (FADD2 / FMUL2 / FFMA2 on
// (re, im) register pairs): a complex add or subtract is one instruction, a complex multiply two.
__device__ __forceinline__ double2 cx_add(double2 a, double2 b) { a.x += b.x; a.y += b.y; return a; }
__device__ __forceinline__ double2 cx_sub(double2 a, double2 b) { a.x -= b.x; a.y -= b.y; return a; }
__device__ __forceinline__ double2 cx_mul(double2 a, double2 b) {
    double2 r; r.x = a.x * b.x - a.y * b.y; r.y = a.x * b.y + a.y * b.x; return r;
}
__device__ __forceinline__ float2 cx_add(float2 a, float2 b) { return __fadd2_rn(a, b); }
__device__ __forceinline__ float2 cx_sub(float2 a, float2 b) { return __ffma2_rn(b, make_float2(-1.f, -1.f), a); }
// a * b = a.x (b.x, b.y) + a.y (-b.y, b.x)
__device__ __forceinline__ float2 cx_mul(float2 a, float2 b) {
    const float2 r = __fmul2_rn(b, make_float2(a.x, a.x));
    return __ffma2_rn(make_float2(-b.y, b.x), make_float2(a.y, a.y), r);
}
__device__ __forceinline__ float2 cx_scale(float2 a, float f) { return __fmul2_rn(a, make_float2(f, f)); }
__device__ __forceinline__ double2 cx_scale(double2 a, double f) { a.x *= f; a.y *= f; return a; }
// d * (c + i s), c and s compile-time constants after unrolling
__device__ __forceinline__ float2 cx_mul_const(float2 d, float c, float s) {
    const float2 r = __fmul2_rn(make_float2(c, s), make_float2(d.x, d.x));
    return __ffma2_rn(make_float2(-s, c), make_float2(d.y, d.y), r);
}
__device__ __forceinline__ double2 cx_mul_const(double2 d, double c, double s) {
    double2 r; r.x = d.x * c - d.y * s; r.y = d.x * s + d.y * c; return r;
}

// d * exp(SIGN * 2 pi i t / 16), t a compile-time constant after unrolling (0 <= t < 8)
template <typename T, int SIGN>
__device__ __forceinline__ Cx<T> mul_w16(Cx<T> d, int t) {
    constexpr double C1 = 0.92387953251128673848, S1 = 0.38268343236508978178, H = 0.70710678118654752440;
    T c, s;
    switch (t) {
        case 0: return d;
        case 4: return SIGN < 0 ? cx_make<T>(d.y, -d.x) : cx_make<T>(-d.y, d.x);
        case 1: c = (T)C1; s = (T)S1; break;
        case 2: c = (T)H; s = (T)H; break;
        case 3: c = (T)S1; s = (T)C1; break;
        case 5: c = (T)-S1; s = (T)C1; break;
        case 6: c = (T)-H; s = (T)H; break;
        default: c = (T)-C1; s = (T)S1; break;
    }
    if (SIGN < 0) s = -s;
    return cx_mul_const(d, c, s);
}

__host__ __device__ constexpr int ilog2(int v) { return v <= 1 ? 0 : 1 + ilog2(v >> 1); }
__host__ __device__ constexpr int bitrev(int i, int bits) {
    int r = 0;
    for (int b = 0; b < bits; ++b) r |= ((i >> b) & 1) << (bits - 1 - b);
    return r;
}

// In-register DFT of R = 2, 4, 8 or 16 points, natural order in and out.
template <typename T, int R, int SIGN>
__device__ __forceinline__ void dft_reg(Cx<T>* v) {
    constexpr int LOG = ilog2(R);
#pragma unroll
    for (int s = 0; s < LOG; ++s) {
        const int len = R >> s;
#pragma unroll
        for (int i = 0; i < R; i += len) {
#pragma unroll
            for (int j = 0; j < len / 2; ++j) {
                Cx<T> a = v[i + j], b = v[i + j + len / 2];
                v[i + j] = cx_add(a, b);
                v[i + j + len / 2] = mul_w16<T, SIGN>(cx_sub(a, b), j * (16 / len));
            }
        }
    }
#pragma unroll
    for (int i = 0; i < R; ++i) {
        const int r = bitrev(i, LOG);
        if (i < r) { Cx<T> t = v[i]; v[i] = v[r]; v[r] = t; }
    }
}

template <int N, int SIGN>
struct FftShape {
    static constexpr int RA = SIGN < 0 ? 16 : N / 16;
    static constexpr int RB = N / RA;
    static constexpr int TPL = N / 16;                 // threads per line
    static constexpr int ITEMS_A = RB / TPL;           // fwd 1, inv 256/N
    static constexpr int ITEMS_B = RA / TPL;           // fwd 256/N, inv 1
    static constexpr int LSP_RAW = RA * (RB + 1);
    static constexpr int LSP = LSP_RAW | 1;            // odd line pitch in shared memory
};
constexpr int kFftThreads = 256;
template <int N> constexpr int fft_lines_per_cta() { return kFftThreads / (N / 16); }
template <typename T, int N> constexpr size_t fft_smem_bytes() {
    // both directions use the same pitch bound: max(16*(N/16+1), (N/16)*17) | 1
    constexpr int a = FftShape<N, -1>::LSP, b = FftShape<N, +1>::LSP;
    return sizeof(Cx<T>) * (size_t)fft_lines_per_cta<N>() * (a > b ? a : b);
}
template <int N> constexpr int fft_line_pitch() {
    return FftShape<N, -1>::LSP > FftShape<N, +1>::LSP ? FftShape<N, -1>::LSP : FftShape<N, +1>::LSP;
}

// Pass A.  v[i*RA + n1] holds x[RB*n1 + a] for item a = t + TPL*i.  Result goes to the
// line's shared buffer at k1*(RB+1) + a.  tw[(SIGN<0 ? 0 : N) + k1*RB + a] = exp(-2 pi i a k1 / N).
template <typename T, int N, int SIGN>
__device__ __forceinline__ void fft_pass_a(Cx<T>* v, int t, Cx<T>* line, const Cx<T>* __restrict__ tw) {
    using S = FftShape<N, SIGN>;
#pragma unroll
    for (int i = 0; i < S::ITEMS_A; ++i) {
        const int a = t + S::TPL * i;
        dft_reg<T, S::RA, SIGN>(v + i * S::RA);
#pragma unroll
        for (int k1 = 0; k1 < S::RA; ++k1) {
            Cx<T> val = v[i * S::RA + k1];
            if (k1 > 0) {
                // table laid out [direction][k1][a]: the lanes of a line (consecutive a) read consecutive
                // entries -- 4 sectors per request instead of ~13 for the a*k1-indexed table
                Cx<T> w = __ldg(&tw[(SIGN < 0 ? 0 : N) + k1 * S::RB + a]);
                if (SIGN > 0) w.y = -w.y;
                val = cx_mul(val, w);
            }
            line[k1 * (S::RB + 1) + a] = val;
        }
    }
}

// Pass B.  After it v[i*RB + k2] holds X[k1 + RA*k2] for k1 = t + TPL*i.
template <typename T, int N, int SIGN>
__device__ __forceinline__ void fft_pass_b(Cx<T>* v, int t, const Cx<T>* line) {
    using S = FftShape<N, SIGN>;
#pragma unroll
    for (int i = 0; i < S::ITEMS_B; ++i) {
        const int k1 = t + S::TPL * i;
#pragma unroll
        for (int a = 0; a < S::RB; ++a) v[i * S::RB + a] = line[k1 * (S::RB + 1) + a];
        dft_reg<T, S::RB, SIGN>(v + i * S::RB);
    }
}

struct FftGeom {
    int n;       // line length = grid points per dimension
    int kcut;
    int Kxp;     // padded count of kept kx
    int Ky;      // 2*kcut + 1
};

// ---------------------------------------------------------------- X passes (contiguous lines)
// Real-to-complex, two rows per transform: z = x1 + i x2, then X1[k] = (Z[k] + conj Z[N-k])/2 and
// X2[k] = (Z[k] - conj Z[N-k])/(2i).  Z[N-k] lives in another thread of the line, so the spectrum
// goes through the line's shared buffer once more (a line's threads are lanes of one warp).
template <typename T, int N>
__global__ void __launch_bounds__(kFftThreads)
fft_x_forward_kernel(const T* __restrict__ G, Cx<T>* __restrict__ A1, FftGeom fg, const Cx<T>* __restrict__ tw) {
    pdl_prologue();
    using S = FftShape<N, -1>;
    static_assert(S::TPL <= 32, "a line must fit in one warp");
    constexpr int LPC = fft_lines_per_cta<N>(), PITCH = fft_line_pitch<N>();
    static_assert(PITCH >= N, "line buffer holds a full spectrum");
    extern __shared__ __align__(16) unsigned char smem_raw[];
    Cx<T>* sm = reinterpret_cast<Cx<T>*>(smem_raw);
    const int t = threadIdx.x % S::TPL, ls = threadIdx.x / S::TPL;
    const size_t row = 2 * ((size_t)blockIdx.x * LPC + ls);    // rows (row, row+1); n*n is a multiple of 2*LPC
    Cx<T> v[16];
    const T* in0 = G + row * N;
    const T* in1 = in0 + N;
#pragma unroll
    for (int n1 = 0; n1 < 16; ++n1) v[n1] = cx_make<T>(in0[S::RB * n1 + t], in1[S::RB * n1 + t]);
    Cx<T>* line = sm + ls * PITCH;
    fft_pass_a<T, N, -1>(v, t, line, tw);
    __syncthreads();
    fft_pass_b<T, N, -1>(v, t, line);
    __syncwarp();                                              // every lane of the line has read pass A's data
#pragma unroll
    for (int i = 0; i < S::ITEMS_B; ++i)
#pragma unroll
        for (int k2 = 0; k2 < S::RB; ++k2) line[t + S::TPL * i + 16 * k2] = v[i * S::RB + k2];
    __syncwarp();
    Cx<T>* out0 = A1 + row * fg.Kxp;
    Cx<T>* out1 = out0 + fg.Kxp;
    const T half = (T)0.5;
#pragma unroll
    for (int i = 0; i < S::ITEMS_B; ++i)
#pragma unroll
        for (int k2 = 0; k2 < S::RB; ++k2) {
            const int k = t + S::TPL * i + 16 * k2;
            if (k < fg.Kxp) {
                Cx<T> x1 = cx_make<T>((T)0, (T)0), x2 = x1;
                if (k <= fg.kcut) {
                    // X1 = (Z[k] + conj Z[N-k])/2,  X2 = -i (Z[k] - conj Z[N-k])/2
                    const Cx<T> zk = v[i * S::RB + k2], zn = line[(N - k) & (N - 1)];
                    const Cx<T> zc = cx_make<T>(zn.x, -zn.y);
                    const Cx<T> sum = cx_add(zk, zc), dif = cx_sub(zk, zc);
                    x1 = cx_scale(sum, half);
                    x2 = cx_scale(cx_make<T>(dif.y, -dif.x), half);
                }
                out0[k] = x1;
                out1[k] = x2;
            }
        }
}

// Complex-to-real, two rows per transform: with Z = X1 + i X2 (X1, X2 the Hermitian spectra of two
// real rows) one complex inverse FFT returns row 1 in the real and row 2 in the imaginary part.
template <typename T, int N>
__global__ void __launch_bounds__(kFftThreads)
fft_x_inverse_kernel(const Cx<T>* __restrict__ A1, T* __restrict__ G, FftGeom fg, const Cx<T>* __restrict__ tw) {
    pdl_prologue();
    using S = FftShape<N, +1>;
    constexpr int LPC = fft_lines_per_cta<N>(), PITCH = fft_line_pitch<N>();
    extern __shared__ __align__(16) unsigned char smem_raw[];
    Cx<T>* sm = reinterpret_cast<Cx<T>*>(smem_raw);
    const int t = threadIdx.x % S::TPL, ls = threadIdx.x / S::TPL;
    const size_t row = 2 * ((size_t)blockIdx.x * LPC + ls);    // rows (row, row+1); n*n is a multiple of 2*LPC
    const Cx<T>* in0 = A1 + row * fg.Kxp;
    const Cx<T>* in1 = in0 + fg.Kxp;
    Cx<T> v[16];
    // Hermitian extension of the half spectra: X[N-k] = conj X[k];  Z = X1 + i X2
#pragma unroll
    for (int i = 0; i < S::ITEMS_A; ++i)
#pragma unroll
        for (int n1 = 0; n1 < S::RA; ++n1) {
            const int e = 16 * n1 + t + S::TPL * i;
            Cx<T> val = cx_make<T>((T)0, (T)0);
            if (e <= fg.kcut) {
                const Cx<T> a = in0[e], b = in1[e];
                val = cx_make<T>(a.x - b.y, a.y + b.x);
            } else if (N - e <= fg.kcut) {
                const Cx<T> a = in0[N - e], b = in1[N - e];       // conj(a) + i conj(b)
                val = cx_make<T>(a.x + b.y, b.x - a.y);
            }
            v[i * S::RA + n1] = val;
        }
    Cx<T>* line = sm + ls * PITCH;
    fft_pass_a<T, N, +1>(v, t, line, tw);
    __syncthreads();
    fft_pass_b<T, N, +1>(v, t, line);
    T* out0 = G + row * N;
    T* out1 = out0 + N;
#pragma unroll
    for (int k2 = 0; k2 < 16; ++k2) { out0[t + S::TPL * k2] = v[k2].x; out1[t + S::TPL * k2] = v[k2].y; }
}

// ---------------------------------------------------------------- X passes, rows staged through TMA
// Persistent variants of the two X passes: a CTA walks tiles (LPC lines = 2 LPC rows, contiguous in memory)
// blockIdx.x, blockIdx.x + gridDim.x, ...  The rows of a tile are brought into shared memory by the TMA
// unit (cp.async.bulk, one 1-D bulk copy per line = two rows, completion on an mbarrier; the line pitch in
// shared memory is padded by 64 bytes so that the two lines a warp reads fall in different banks).  There
// is ONE staging buffer: as soon as every thread has taken its tile out of it into registers, the copy of
// the CTA's next tile is issued, so it runs under the whole transform + store of the current tile.
// global -> shared bulk copy (TMA, 1-D): bytes is a multiple of 16, both addresses 16-byte aligned
__device__ __forceinline__ void tma_load_1d(void* smem_dst, const void* gmem_src, uint32_t bytes, uint64_t* bar) {
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];"
                 ::"r"(smem_u32(smem_dst)), "l"(gmem_src), "r"(bytes), "r"(smem_u32(bar)) : "memory");
}

template <typename T, int N> constexpr int fft_xf_stage_pitch() { return 2 * N + 64 / (int)sizeof(T); }      // in T
template <typename T, int N> constexpr size_t fft_xf_tma_smem_bytes() {
    return fft_smem_bytes<T, N>() + sizeof(T) * (size_t)fft_lines_per_cta<N>() * fft_xf_stage_pitch<T, N>() + 16;
}

template <typename T, int N>
__global__ void __launch_bounds__(kFftThreads)
fft_x_forward_tma_kernel(const T* __restrict__ G, Cx<T>* __restrict__ A1, FftGeom fg, const Cx<T>* __restrict__ tw,
                         int ntiles) {
    pdl_prologue();
    using S = FftShape<N, -1>;
    static_assert(S::TPL <= 32, "a line must fit in one warp");
    constexpr int LPC = fft_lines_per_cta<N>(), PITCH = fft_line_pitch<N>(), SP = fft_xf_stage_pitch<T, N>();
    constexpr uint32_t LINE_BYTES = 2 * N * sizeof(T);
    extern __shared__ __align__(16) unsigned char smem_raw[];
    Cx<T>* sm = reinterpret_cast<Cx<T>*>(smem_raw);
    T* stage = reinterpret_cast<T*>(smem_raw + fft_smem_bytes<T, N>());
    uint64_t* bar = reinterpret_cast<uint64_t*>(stage + (size_t)LPC * SP);
    const int t = threadIdx.x % S::TPL, ls = threadIdx.x / S::TPL;
    if (threadIdx.x == 0) {
        mbar_init(bar, 1);
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    __syncthreads();
    // producer side: thread 0 arms the barrier with the tile's bytes, the first thread of every line copies it
    auto issue = [&](int tile) {
        if (threadIdx.x == 0) mbar_expect_tx(bar, LINE_BYTES * LPC);
        __syncthreads();                                    // the expectation is armed before any copy can complete
        if (t == 0) tma_load_1d(stage + (size_t)ls * SP, G + (2 * ((size_t)tile * LPC + ls)) * N, LINE_BYTES, bar);
    };
    int tile = blockIdx.x;
    if (tile < ntiles) issue(tile);
    uint32_t parity = 0;
    const T half = (T)0.5;
    for (; tile < ntiles; tile += gridDim.x) {
        mbar_wait(bar, parity);
        parity ^= 1u;
        const size_t row = 2 * ((size_t)tile * LPC + ls);
        Cx<T> v[16];
        const T* in0 = stage + (size_t)ls * SP;
        const T* in1 = in0 + N;
#pragma unroll
        for (int n1 = 0; n1 < 16; ++n1) v[n1] = cx_make<T>(in0[S::RB * n1 + t], in1[S::RB * n1 + t]);
        __syncthreads();                                    // every thread holds its tile: the buffer is free
        if (tile + (int)gridDim.x < ntiles) issue(tile + gridDim.x);
        Cx<T>* line = sm + ls * PITCH;
        fft_pass_a<T, N, -1>(v, t, line, tw);
        __syncthreads();
        fft_pass_b<T, N, -1>(v, t, line);
        __syncwarp();
#pragma unroll
        for (int i = 0; i < S::ITEMS_B; ++i)
#pragma unroll
            for (int k2 = 0; k2 < S::RB; ++k2) line[t + S::TPL * i + 16 * k2] = v[i * S::RB + k2];
        __syncwarp();
        Cx<T>* out0 = A1 + row * fg.Kxp;
        Cx<T>* out1 = out0 + fg.Kxp;
#pragma unroll
        for (int i = 0; i < S::ITEMS_B; ++i)
#pragma unroll
            for (int k2 = 0; k2 < S::RB; ++k2) {
                const int k = t + S::TPL * i + 16 * k2;
                if (k < fg.Kxp) {
                    Cx<T> x1 = cx_make<T>((T)0, (T)0), x2 = x1;
                    if (k <= fg.kcut) {
                        const Cx<T> zk = v[i * S::RB + k2], zn = line[(N - k) & (N - 1)];
                        const Cx<T> zc = cx_make<T>(zn.x, -zn.y);
                        const Cx<T> sum = cx_add(zk, zc), dif = cx_sub(zk, zc);
                        x1 = cx_scale(sum, half);
                        x2 = cx_scale(cx_make<T>(dif.y, -dif.x), half);
                    }
                    out0[k] = x1;
                    out1[k] = x2;
                }
            }
        __syncthreads();                                    // the line buffers are rewritten by the next tile
    }
}

// X inverse (complex-to-real) with the half-spectrum rows staged through TMA; same structure as above.
// A line = the two consecutive rows (row, row + 1) of A1 = 2 Kxp complex values, contiguous.
template <typename T> constexpr int fft_xi_stage_pad() { return 16 / (int)sizeof(Cx<T>) * 2; }    // complex values
template <typename T, int N> size_t fft_xi_tma_smem_bytes(int Kxp) {
    return fft_smem_bytes<T, N>() + sizeof(Cx<T>) * (size_t)fft_lines_per_cta<N>() * (2 * Kxp + fft_xi_stage_pad<T>()) + 16;
}

template <typename T, int N>
__global__ void __launch_bounds__(kFftThreads)
fft_x_inverse_tma_kernel(const Cx<T>* __restrict__ A1, T* __restrict__ G, FftGeom fg, const Cx<T>* __restrict__ tw,
                         int ntiles) {
    pdl_prologue();
    using S = FftShape<N, +1>;
    constexpr int LPC = fft_lines_per_cta<N>(), PITCH = fft_line_pitch<N>();
    extern __shared__ __align__(16) unsigned char smem_raw[];
    Cx<T>* sm = reinterpret_cast<Cx<T>*>(smem_raw);
    Cx<T>* stage = reinterpret_cast<Cx<T>*>(smem_raw + fft_smem_bytes<T, N>());
    const int SP = 2 * fg.Kxp + fft_xi_stage_pad<T>();                       // line pitch in complex values
    const uint32_t LINE_BYTES = 2u * (uint32_t)fg.Kxp * (uint32_t)sizeof(Cx<T>);
    uint64_t* bar = reinterpret_cast<uint64_t*>(stage + (size_t)LPC * SP);
    const int t = threadIdx.x % S::TPL, ls = threadIdx.x / S::TPL;
    if (threadIdx.x == 0) {
        mbar_init(bar, 1);
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    __syncthreads();
    auto issue = [&](int tile) {
        if (threadIdx.x == 0) mbar_expect_tx(bar, LINE_BYTES * LPC);
        __syncthreads();
        if (t == 0) tma_load_1d(stage + (size_t)ls * SP, A1 + (2 * ((size_t)tile * LPC + ls)) * fg.Kxp, LINE_BYTES, bar);
    };
    int tile = blockIdx.x;
    if (tile < ntiles) issue(tile);
    uint32_t parity = 0;
    for (; tile < ntiles; tile += gridDim.x) {
        mbar_wait(bar, parity);
        parity ^= 1u;
        const size_t row = 2 * ((size_t)tile * LPC + ls);
        const Cx<T>* in0 = stage + (size_t)ls * SP;
        const Cx<T>* in1 = in0 + fg.Kxp;
        Cx<T> v[16];
        // Hermitian extension of the half spectra: X[N-k] = conj X[k];  Z = X1 + i X2
#pragma unroll
        for (int i = 0; i < S::ITEMS_A; ++i)
#pragma unroll
            for (int n1 = 0; n1 < S::RA; ++n1) {
                const int e = 16 * n1 + t + S::TPL * i;
                Cx<T> val = cx_make<T>((T)0, (T)0);
                if (e <= fg.kcut) {
                    const Cx<T> a = in0[e], b = in1[e];
                    val = cx_make<T>(a.x - b.y, a.y + b.x);
                } else if (N - e <= fg.kcut) {
                    const Cx<T> a = in0[N - e], b = in1[N - e];       // conj(a) + i conj(b)
                    val = cx_make<T>(a.x + b.y, b.x - a.y);
                }
                v[i * S::RA + n1] = val;
            }
        __syncthreads();                                    // every thread holds its tile: the buffer is free
        if (tile + (int)gridDim.x < ntiles) issue(tile + gridDim.x);
        Cx<T>* line = sm + ls * PITCH;
        fft_pass_a<T, N, +1>(v, t, line, tw);
        __syncthreads();
        fft_pass_b<T, N, +1>(v, t, line);
        T* out0 = G + row * N;
        T* out1 = out0 + N;
#pragma unroll
        for (int k2 = 0; k2 < 16; ++k2) { out0[t + S::TPL * k2] = v[k2].x; out1[t + S::TPL * k2] = v[k2].y; }
        __syncthreads();                                    // the line buffers are rewritten by the next tile
    }
}

// ---------------------------------------------------------------- Y passes (strided lines)
// line id = z*Kxp + kx; consecutive ids are contiguous in memory.
template <typename T, int N>
__global__ void __launch_bounds__(kFftThreads)
fft_y_forward_kernel(const Cx<T>* __restrict__ A1, Cx<T>* __restrict__ A2, FftGeom fg, const Cx<T>* __restrict__ tw) {
    pdl_prologue();
    using S = FftShape<N, -1>;
    constexpr int LPC = fft_lines_per_cta<N>(), PITCH = fft_line_pitch<N>();
    extern __shared__ __align__(16) unsigned char smem_raw[];
    Cx<T>* sm = reinterpret_cast<Cx<T>*>(smem_raw);
    const int ls = threadIdx.x % LPC, t = threadIdx.x / LPC;
    const size_t id = (size_t)blockIdx.x * LPC + ls;           // n*Kxp is a multiple of LPC? guarded below
    const size_t total = (size_t)N * fg.Kxp;
    const bool live = id < total;
    const int z = live ? (int)(id / fg.Kxp) : 0, kx = live ? (int)(id % fg.Kxp) : 0;
    const Cx<T>* in = A1 + (size_t)z * N * fg.Kxp + kx;
    Cx<T> v[16];
#pragma unroll
    for (int n1 = 0; n1 < 16; ++n1)
        v[n1] = live ? in[(unsigned)(S::RB * n1 + t) * (unsigned)fg.Kxp] : cx_make<T>((T)0, (T)0);
    Cx<T>* line = sm + ls * PITCH;
    fft_pass_a<T, N, -1>(v, t, line, tw);
    __syncthreads();
    fft_pass_b<T, N, -1>(v, t, line);
    if (!live) return;
    Cx<T>* out = A2 + (size_t)z * fg.Ky * fg.Kxp + kx;
#pragma unroll
    for (int i = 0; i < S::ITEMS_B; ++i)
#pragma unroll
        for (int k2 = 0; k2 < S::RB; ++k2) {
            const int k = t + S::TPL * i + 16 * k2;
            int kyp = -1;
            if (k <= fg.kcut) kyp = k;
            else if (k >= N - fg.kcut) kyp = k - N + fg.Ky;
            if (kyp >= 0) out[(unsigned)kyp * (unsigned)fg.Kxp] = v[i * S::RB + k2];
        }
}

template <typename T, int N>
__global__ void __launch_bounds__(kFftThreads)
fft_y_inverse_kernel(const Cx<T>* __restrict__ A2, Cx<T>* __restrict__ A1, FftGeom fg, const Cx<T>* __restrict__ tw) {
    pdl_prologue();
    using S = FftShape<N, +1>;
    constexpr int LPC = fft_lines_per_cta<N>(), PITCH = fft_line_pitch<N>();
    extern __shared__ __align__(16) unsigned char smem_raw[];
    Cx<T>* sm = reinterpret_cast<Cx<T>*>(smem_raw);
    const int ls = threadIdx.x % LPC, t = threadIdx.x / LPC;
    const size_t id = (size_t)blockIdx.x * LPC + ls;
    const size_t total = (size_t)N * fg.Kxp;
    const bool live = id < total;
    const int z = live ? (int)(id / fg.Kxp) : 0, kx = live ? (int)(id % fg.Kxp) : 0;
    const Cx<T>* in = A2 + (size_t)z * fg.Ky * fg.Kxp + kx;
    Cx<T> v[16];
#pragma unroll
    for (int i = 0; i < S::ITEMS_A; ++i)
#pragma unroll
        for (int n1 = 0; n1 < S::RA; ++n1) {
            const int e = 16 * n1 + t + S::TPL * i;
            int kyp = -1;
            if (e <= fg.kcut) kyp = e;
            else if (e >= N - fg.kcut) kyp = e - N + fg.Ky;
            v[i * S::RA + n1] = (live && kyp >= 0) ? in[(unsigned)kyp * (unsigned)fg.Kxp] : cx_make<T>((T)0, (T)0);
        }
    Cx<T>* line = sm + ls * PITCH;
    fft_pass_a<T, N, +1>(v, t, line, tw);
    __syncthreads();
    fft_pass_b<T, N, +1>(v, t, line);
    if (!live) return;
    Cx<T>* out = A1 + (size_t)z * N * fg.Kxp + kx;
#pragma unroll
    for (int k2 = 0; k2 < 16; ++k2) out[(unsigned)(t + S::TPL * k2) * (unsigned)fg.Kxp] = v[k2];
}

// ---------------------------------------------------------------- fused Z pass
// For every kept (kx, ky) line: forward FFT along z, then for each kz with
// 0 < kx^2+ky^2+kz^2 <= k_cut^2 (R4, R12)
//     S~ = g^ * iphi[kx] iphi[|ky|] iphi[|kz|]          (scaling, 1/D)
//     E += mult * wf[|k|^2] |S~|^2                      (Eq. 38; mult = 2 for kx > 0: Hermitian half)
//     psi^ = wf[|k|^2] * S~ * iphi iphi iphi            (subdividing; zero outside the sphere)
// and the inverse FFT along z, in place.  wf[s] = f(s)^2 w(s) (Slater factor folded in, R19).
// NOUT = 1: analytic variant (psi^).  NOUT = 3: ik variant, b^_d = -i n_d psi^ into out0..2.
struct ScaleTables {
    const void* iphi;   // [kcut+1]   1/Phi(k)
    const void* wf;     // [kcut^2+1] f^2 w, entry 0 unused (= 0)
};
// Orthorhombic plans (kBox; R26): the weight is not a function of the integer |n|^2, so it is evaluated
// in place, in fp64, from s = |h|^2 Lmax^2 = nx^2 (Lmax/Lx)^2 + ny^2 (Lmax/Ly)^2 + nz^2 (Lmax/Lz)^2 (each product and
// sum rounded once, in this order: membership s <= k_cut^2 is decided on this number):
//   w = f^2 exp(-pi^2 |h|^2/alpha^2)/|h|^2,  f^2 = (1 + pi^2 lambda^2 |h|^2)^-4,  |h|^2 = s/Lmax^2    (length^2)
// rounded once to T like the tables.  ik variant: b^_d = -i h_d psi^, h_d = n_d / L_d.
struct BoxScale {
    double a[3];        // (Lmax/L_d)^2
    double l[3];        // L_d
    double lm2;         // Lmax^2
    double alpha, lambda;
};

// Step a7 inside the Z pass: every CTA publishes its fp64 energy partial (thread 0's `mine`); the CTA that
// finishes last sums all partials in a fixed order (strided per thread, then a tree: the same order whichever
// CTA it is, so E is reproducible) and writes E = scale * sum.  The counter resets itself for the next call.
// Must be called by all threads of the CTA.
__device__ __forceinline__ void z_pass_energy_finish(double mine, double* __restrict__ e_partial,
                                                     unsigned* __restrict__ done_count, double e_scale,
                                                     double* __restrict__ e_out) {
    __shared__ bool is_last;
    __shared__ double fin[kFftThreads];
    if (threadIdx.x == 0) {
        e_partial[blockIdx.x] = mine;
        __threadfence();
        is_last = atomicAdd(done_count, 1u) == gridDim.x - 1;
    }
    __syncthreads();
    if (!is_last) return;
    __threadfence();
    double s = 0.0;
    for (unsigned i = threadIdx.x; i < gridDim.x; i += kFftThreads) s += __ldcg(&e_partial[i]);
    fin[threadIdx.x] = s;
    __syncthreads();
    for (int o = kFftThreads / 2; o > 0; o >>= 1) {
        if ((int)threadIdx.x < o) fin[threadIdx.x] += fin[threadIdx.x + o];
        __syncthreads();
    }
    if (threadIdx.x == 0) { *e_out = e_scale * fin[0]; *done_count = 0u; }
}

template <typename T, int N, int NOUT, bool kBox = false>
__global__ void __launch_bounds__(kFftThreads)
fft_z_fused_kernel(Cx<T>* __restrict__ A2, Cx<T>* __restrict__ out1, Cx<T>* __restrict__ out2, FftGeom fg,
                   const Cx<T>* __restrict__ tw, ScaleTables st, double* __restrict__ e_partial,
                   Cx<T>* __restrict__ spectrum, unsigned* __restrict__ done_count, double e_scale,
                   double* __restrict__ e_out, const BoxScale bs) {
    pdl_prologue();
    using SF = FftShape<N, -1>;
    using SI = FftShape<N, +1>;
    constexpr int LPC = fft_lines_per_cta<N>(), PITCH = fft_line_pitch<N>();
    extern __shared__ __align__(16) unsigned char smem_raw[];
    Cx<T>* sm = reinterpret_cast<Cx<T>*>(smem_raw);
    __shared__ double red[kFftThreads / 32];
    const T* iphi = static_cast<const T*>(st.iphi);
    const T* wf = static_cast<const T*>(st.wf);

    const int ls = threadIdx.x % LPC, t = threadIdx.x / LPC;
    const size_t id = (size_t)blockIdx.x * LPC + ls;
    const size_t total = (size_t)fg.Ky * fg.Kxp;
    const bool live = id < total;
    const int kyp = live ? (int)(id / fg.Kxp) : 0, kx = live ? (int)(id % fg.Kxp) : 0;
    const int ky = kyp <= fg.kcut ? kyp : kyp - fg.Ky;
    const int kc2 = fg.kcut * fg.kcut;
    const int kxy2 = kx * kx + ky * ky;
    const double sxy = kBox ? __dadd_rn(__dmul_rn((double)(kx * kx), bs.a[0]), __dmul_rn((double)(ky * ky), bs.a[1])) : 0.0;
    const bool inside = live && kx <= fg.kcut && (kBox ? sxy <= (double)kc2 : kxy2 <= kc2);
    const unsigned zstride = (unsigned)fg.Ky * (unsigned)fg.Kxp;   // all offsets fit 32 bits (<= 2^23 elements)
    Cx<T>* base = A2 + (size_t)kyp * fg.Kxp + kx;
    const Cx<T> zero = cx_make<T>((T)0, (T)0);

    // whole CTA outside the cylinder kx^2+ky^2 <= kcut^2: the field spectrum is zero there
    if (!__syncthreads_or(inside)) {
        if (live) {
#pragma unroll
            for (int n1 = 0; n1 < 16; ++n1) {
                const unsigned o = (unsigned)(SF::RB * n1 + t) * zstride;
                base[o] = zero;
                if (NOUT == 3) { out1[(base - A2) + o] = zero; out2[(base - A2) + o] = zero; }
            }
        }
        z_pass_energy_finish(0.0, e_partial, done_count, e_scale, e_out);
        return;
    }

    Cx<T> v[16];
#pragma unroll
    for (int n1 = 0; n1 < 16; ++n1)
        v[n1] = inside ? base[(unsigned)(SF::RB * n1 + t) * zstride] : zero;
    Cx<T>* line = sm + ls * PITCH;
    fft_pass_a<T, N, -1>(v, t, line, tw);
    __syncthreads();
    fft_pass_b<T, N, -1>(v, t, line);
    __syncthreads();    // shared buffer is reused by the inverse transform

    double e_acc = 0.0;
    const T ipxy = inside ? iphi[kx] * iphi[ky < 0 ? -ky : ky] : (T)0;
    const double mult = kx > 0 ? 2.0 : 1.0;
    int kzs[16];
#pragma unroll
    for (int i = 0; i < SF::ITEMS_B; ++i)
#pragma unroll
        for (int k2 = 0; k2 < SF::RB; ++k2) {
            const int r = i * SF::RB + k2;
            const int k = t + SF::TPL * i + 16 * k2;
            const int kz = k < N / 2 ? k : k - N;
            kzs[r] = kz;
            const int akz = kz < 0 ? -kz : kz;
            const int s = kxy2 + kz * kz;
            bool in_k = inside && akz <= fg.kcut && s > 0;
            T w = (T)0;
            if constexpr (kBox) {
                const double sb = __dadd_rn(sxy, __dmul_rn((double)(kz * kz), bs.a[2]));
                in_k = in_k && sb <= (double)kc2;
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
                const T ip3 = ipxy * iphi[akz];
                Cx<T> S = cx_make<T>(v[r].x * ip3, v[r].y * ip3);
                e_acc += mult * (double)w * ((double)S.x * (double)S.x + (double)S.y * (double)S.y);
                if (spectrum) {
                    const int kzp = kz >= 0 ? kz : kz + fg.Ky;
                    spectrum[((size_t)kzp * fg.Ky + kyp) * fg.Kxp + kx] = S;
                }
                const T sc = w * ip3;
                v[r] = cx_make<T>(S.x * sc, S.y * sc);
            } else {
                v[r] = zero;
            }
        }

    Cx<T>* outs[3] = {A2, out1, out2};
    Cx<T> keep[NOUT == 3 ? 16 : 1];
    if (NOUT == 3) {
#pragma unroll
        for (int r = 0; r < 16; ++r) keep[r] = v[r];
    }
#pragma unroll
    for (int d = 0; d < NOUT; ++d) {
        if (NOUT == 3) {
            // b^_d = -i n_d psi^ :  -i (x + i y) = y - i x
#pragma unroll
            for (int r = 0; r < 16; ++r) {
                const int ni = d == 0 ? kx : (d == 1 ? ky : kzs[r]);
                const T nd = kBox ? (T)((double)ni / bs.l[d]) : (T)ni;
                v[r] = cx_make<T>(nd * keep[r].y, -nd * keep[r].x);
            }
            if (d > 0) __syncthreads();
        }
        fft_pass_a<T, N, +1>(v, t, line, tw);
        __syncthreads();
        fft_pass_b<T, N, +1>(v, t, line);
        if (live) {
            Cx<T>* ob = outs[d] + (size_t)kyp * fg.Kxp + kx;
#pragma unroll
            for (int k2 = 0; k2 < 16; ++k2) ob[(unsigned)(t + SI::TPL * k2) * zstride] = v[k2];
        }
    }

    // deterministic block reduction of the fp64 energy partial
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) e_acc += __shfl_xor_sync(0xffffffffu, e_acc, o);
    if ((threadIdx.x & 31) == 0) red[threadIdx.x >> 5] = e_acc;
    __syncthreads();
    double s = 0.0;
    if (threadIdx.x == 0) {
#pragma unroll
        for (int w = 0; w < kFftThreads / 32; ++w) s += red[w];
    }
    z_pass_energy_finish(s, e_partial, done_count, e_scale, e_out);
}


}  // namespace enuf
