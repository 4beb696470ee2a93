// Step a6 -- interpolating (forward NFFT, last part; Eq. 42 :340).
//
// One CTA per 16^3 grid tile, working on the tile's particles (a contiguous range of 16
// bins, TileGeom), with the tile plus a halo of m cells per side ((16+2m)^3 values) held in
// shared memory.  Particles are taken in batches: first the 3 W window values and
// derivatives of every particle of the batch are computed once (one thread per particle and
// dimension) and kept on chip, then one warp per particle contracts the
// (2m+1)^3 stencil: every lane owns x-rows of the stencil (row strides chosen so that the 32
// rows a warp reads at once fall in 32 different banks), forms s = sum_x Psi (phi, phi') with
// packed FMAs, and the three force components come out of one pass over the field
// ("forces in 3D packed into a single calculation entity").
#pragma once

#include "enuf_common.cuh"
#include "enuf_spread.cuh"   // Pair2, fma_pair

namespace enuf {

template <int M_> struct GatherStride;   // (row stride, plane stride) of the shared tile: conflict-free
template <> struct GatherStride<1> { static constexpr int SX = 18, SPL = 325; };
template <> struct GatherStride<2> { static constexpr int SX = 21, SPL = 425; };
template <> struct GatherStride<3> { static constexpr int SX = 23, SPL = 513; };
template <> struct GatherStride<4> { static constexpr int SX = 25, SPL = 609; };
template <> struct GatherStride<5> { static constexpr int SX = 27, SPL = 713; };
template <> struct GatherStride<6> { static constexpr int SX = 29, SPL = 825; };

template <int M_>
struct GatherCfg {
    static constexpr int W = 2 * M_ + 1;
    static constexpr int TP = kTile + 2 * M_;                   // padded tile edge
    static constexpr int SX = GatherStride<M_>::SX;
    static constexpr int SPL = GatherStride<M_>::SPL;
    static constexpr int CELLS = ((TP * SPL + 3) / 4) * 4;      // shared tile size in elements (16 B multiple)
    static constexpr int WARPS = 8;
    static constexpr int NT = WARPS * 32;
    static constexpr int PB = 32;                               // particles per batch
    static constexpr int ITER = (W * W + 31) / 32;              // stencil rows per lane
};

template <typename T, int M_>
constexpr size_t gather_smem_bytes() {
    using C = GatherCfg<M_>;
    // tile + per batch: (phi, phi') pairs [PB][3][16] + (q, idx, base offset) per particle
    return sizeof(T) * ((size_t)C::CELLS + (size_t)C::PB * 3 * 16 * 2 + C::PB) + sizeof(int) * 2 * C::PB;
}

// acc += w2 * v  (both halves, scalar v)
__device__ __forceinline__ void fma_pair_s(float2& acc, const float2 w2, const float v) { fma_pair(acc, w2, v); }
__device__ __forceinline__ void fma_pair_s(double2& acc, const double2 w2, const double v) { fma_pair(acc, w2, v); }

// kIk = false: analytic-derivative variant, F = pre*q * sum Psi[l] grad(phi phi phi)
//              with pre = -n/(pi L^2)  (exact gradient of the ENUF energy).
// kIk = true : one component d of the paper's ik variant, F[.,d] = pre*q * sum B_d[l] phi phi phi
//              with pre = 2/L^2 (Eq. 42).
template <typename T, int M_, bool kIk>
__global__ void __launch_bounds__(GatherCfg<M_>::NT)
gather_kernel(const T* __restrict__ field, const PRec<T>* __restrict__ rec,
              const uint32_t* __restrict__ cell, const uint32_t* __restrict__ idx,
              const uint32_t* __restrict__ offset, TileGeom g, WindowParams wp,
              const __grid_constant__ PolyArg<M_> pa, T pre, int component, T* __restrict__ F) {
    using C = GatherCfg<M_>;
    using P2 = typename Pair2<T>::type;
    constexpr int W = C::W, TP = C::TP, SX = C::SX, SPL = C::SPL, NT = C::NT, PB = C::PB, ITER = C::ITER;

    // tile (Tx, Ty, Tz): bins (Ty*nt + Tx)*n + 16 Tz .. + 16
    const int ntz = g.n / kTile;
    const int Tz = blockIdx.x % ntz, col = blockIdx.x / ntz;
    const int Tx = col % g.nt, Ty = col / g.nt;
    const int bin0 = col * g.n + Tz * kTile;
    const uint32_t start = offset[bin0];
    const int cnt = (int)(offset[bin0 + kTile] - start);
    if (cnt == 0) return;

    extern __shared__ __align__(16) unsigned char smem_raw[];
    T* tile_s = reinterpret_cast<T*>(smem_raw);
    P2* wtab = reinterpret_cast<P2*>(tile_s + C::CELLS);        // [PB][3][16] (phi, phi')
    T* q_s = reinterpret_cast<T*>(wtab + PB * 3 * 16);          // [PB] pre * q
    int* base_s = reinterpret_cast<int*>(q_s + PB);             // [PB] tile offset of the stencil origin
    int* idx_s = base_s + PB;                                   // [PB] caller index

    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int tx0 = Tx * kTile, ty0 = Ty * kTile, tz0 = Tz * kTile;

    // ---- stage the padded tile: one row of TP values per warp pass
    for (int rw = warp; rw < TP * TP; rw += C::WARPS) {
        const int lz = rw / TP, ly = rw - lz * TP;
        int gy = ty0 - M_ + ly, gz = tz0 - M_ + lz;
        gy += gy < 0 ? g.n : 0; gy -= gy >= g.n ? g.n : 0;
        gz += gz < 0 ? g.n : 0; gz -= gz >= g.n ? g.n : 0;
        if (lane < TP) {
            int gx = tx0 - M_ + lane;
            gx += gx < 0 ? g.n : 0; gx -= gx >= g.n ? g.n : 0;
            tile_s[lz * SPL + ly * SX + lane] = field[((size_t)gz * g.n + gy) * g.n + gx];
        }
    }

    // stencil rows owned by this lane: rr = lane + 32 it -> (rz, ry)
    int rowoff[ITER], ryo[ITER], rzo[ITER];
#pragma unroll
    for (int it = 0; it < ITER; ++it) {
        const int rr = lane + 32 * it;
        const int rz = rr / W, ry = rr - rz * W;
        rowoff[it] = rz * SPL + ry * SX;
        ryo[it] = 16 + ry;          // index into the particle's [3][16] weight rows
        rzo[it] = 32 + rz;
    }

    for (int b0 = 0; b0 < cnt; b0 += PB) {
        const int nb = min(PB, cnt - b0);
        __syncthreads();        // tile staged / previous batch consumed
        // ---- window values of the batch: one task per (dimension, particle)
        for (int t = tid; t < 3 * nb; t += NT) {
            const int dim = t / nb, slot = t - dim * nb;
            const PRec<T> pr = rec[start + b0 + slot];
            const T d0 = dim == 0 ? pr.dx : (dim == 1 ? pr.dy : pr.dz);
            T w[W], dw[W];
            stencil_weights<T, M_, !kIk>(wp, pa, d0, w, dw);
            P2* row = wtab + (slot * 3 + dim) * 16;
#pragma unroll
            for (int k = 0; k < W; ++k) { P2 v; v.x = w[k]; v.y = dw[k]; row[k] = v; }
            if (dim == 0) {
                int cx, cy, cz;
                unpack_cell(cell[start + b0 + slot], cx, cy, cz);
                base_s[slot] = (cz - tz0) * SPL + (cy - ty0) * SX + (cx - tx0);
                q_s[slot] = pre * pr.q;
                idx_s[slot] = (int)idx[start + b0 + slot];
            }
        }
        __syncthreads();
        // ---- one warp per particle
        for (int slot = warp; slot < nb; slot += C::WARPS) {
            const P2* wt = wtab + slot * 3 * 16;
            P2 wx[W];
#pragma unroll
            for (int k = 0; k < W; ++k) wx[k] = wt[k];
            const T* origin = tile_s + base_s[slot];
            T fx = (T)0, fy = (T)0, fz = (T)0;
#pragma unroll
            for (int it = 0; it < ITER; ++it) {
                if (lane + 32 * it < W * W) {
                    const T* row = origin + rowoff[it];
                    P2 s; s.x = (T)0; s.y = (T)0;
#pragma unroll
                    for (int k = 0; k < W; ++k) fma_pair_s(s, wx[k], row[k]);
                    const P2 wy = wt[ryo[it]], wz = wt[rzo[it]];
                    if (kIk) {
                        fx += s.x * (wy.x * wz.x);
                    } else {
                        fx += s.y * (wy.x * wz.x);
                        fy += s.x * (wy.y * wz.x);
                        fz += s.x * (wy.x * wz.y);
                    }
                }
            }
#pragma unroll
            for (int o = 16; o > 0; o >>= 1) {
                fx += __shfl_xor_sync(0xffffffffu, fx, o);
                if (!kIk) {
                    fy += __shfl_xor_sync(0xffffffffu, fy, o);
                    fz += __shfl_xor_sync(0xffffffffu, fz, o);
                }
            }
            if (lane == 0) {
                const size_t j = (size_t)(uint32_t)idx_s[slot];
                const T sc = q_s[slot];
                if (kIk) {
                    F[3 * j + component] = sc * fx;
                } else {
                    F[3 * j] = sc * fx; F[3 * j + 1] = sc * fy; F[3 * j + 2] = sc * fz;
                }
            }
        }
    }
}

}  // namespace enuf
