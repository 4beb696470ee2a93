// Step a2 -- spreading (adjoint NFFT, part 1):
//   g[l] = sum_j q_j phi(u_jx - l_x) phi(u_jy - l_y) phi(u_jz - l_z), l periodic.
// Step a6 -- interpolating (forward NFFT, last part; Eq. 42 :340).
//
// Both run one CTA per grid tile of TILE^3 cells on the tile's particles (binned by a1),
// with the tile plus a halo of m cells per side ((TILE+2m)^3 values) held in shared memory
// and the 3*(2m+1) window values of a particle computed once per particle and kept on
// chip (the paper's "window values computed in local memory").
//
// Spread -- no shared-memory atomics (fp32 atomicAdd on shared memory is a CAS loop on
// sm_100a).  Instead every shared cell has exactly one owner thread: thread (ty, tz) owns
// all cells with ly = ty (mod W), lz = tz (mod W).  A (2m+1)^2 block of (y, z) rows hits
// every residue pair exactly once, so all W*W threads work on every particle, each doing
// the W cells of one x-row, and the read-modify-write of a cell is always done by the
// same thread in program order: race-free without atomics or barriers, and the summation
// order inside a tile is the sorted particle order.  Only the flush of the padded tile to
// the global grid uses (global) atomic adds, because halos of neighbouring tiles overlap.
#pragma once

#include "enuf_common.cuh"

namespace enuf {

template <int M_, int TILE>
struct TileCfg {
    static constexpr int W = 2 * M_ + 1;
    static constexpr int TP = TILE + 2 * M_;                    // padded tile edge
    static constexpr int SX = (TP % 2 == 0) ? TP + 1 : TP;      // odd row stride (bank spread)
    static constexpr int SPL = TP * SX + ((TP * SX) % 2 == 0 ? 1 : 0) + 2;  // plane stride
    static constexpr int CELLS = ((TP * SPL + 3) / 4) * 4;      // shared tile size in elements (16 B multiple)
    static constexpr int PB = 16;                               // particles per weight batch
    static constexpr int SPREAD_THREADS = ((W * W + 31) / 32) * 32;
    static constexpr int GATHER_WARPS = 8;
};

template <typename T, int M_, int TILE>
constexpr size_t spread_smem_bytes() {
    using C = TileCfg<M_, TILE>;
    return sizeof(T) * ((size_t)C::CELLS + 2 * C::PB * 3 * 16) + sizeof(int) * 2 * C::PB * 4;
}

template <typename T, int M_, int TILE>
__global__ void __launch_bounds__(TileCfg<M_, TILE>::SPREAD_THREADS)
spread_kernel(const PRec<T>* __restrict__ rec, const uint32_t* __restrict__ cell,
              const uint32_t* __restrict__ offset, TileGeom g, WindowParams wp, T* __restrict__ grid) {
    using C = TileCfg<M_, TILE>;
    constexpr int W = C::W, TP = C::TP, SX = C::SX, SPL = C::SPL, PB = C::PB;
    constexpr int NT = C::SPREAD_THREADS;

    const int tile = blockIdx.x;
    const uint32_t start = offset[tile];
    const int cnt = (int)(offset[tile + 1] - start);
    if (cnt == 0) return;

    extern __shared__ __align__(16) unsigned char smem_raw[];
    T* tile_s = reinterpret_cast<T*>(smem_raw);
    T* wtab = tile_s + C::CELLS;                         // [2][PB][3][16]
    int* base_s = reinterpret_cast<int*>(wtab + 2 * PB * 3 * 16);   // [2][PB][4]

    const int tid = threadIdx.x;
    for (int e = tid; e < C::CELLS; e += NT) tile_s[e] = (T)0;

    const int tx0 = (tile % g.nt) * TILE, ty0 = ((tile / g.nt) % g.nt) * TILE, tz0 = (tile / (g.nt * g.nt)) * TILE;
    const int ty = tid % W, tz = tid / W;               // owned residues (tid < W*W)
    constexpr int KW = ((TILE + W - 1) / W) * W;        // multiple of W >= TILE

    int buf = 0;
    for (int b0 = 0; b0 < cnt; b0 += PB, buf ^= 1) {
        const int nb = min(PB, cnt - b0);
        T* wt = wtab + buf * (PB * 3 * 16);
        int* bs = base_s + buf * (PB * 4);
        // window values of the batch, once per particle (q folded into the x weights)
        for (int e = tid; e < nb * 3 * W; e += NT) {
            int p = e / (3 * W), rem = e - p * 3 * W, dim = rem / W, k = rem - dim * W;
            const PRec<T> pr = rec[start + b0 + p];
            T d0 = dim == 0 ? pr.dx : (dim == 1 ? pr.dy : pr.dz);
            T phi, dphi;
            window_eval<T, false>(wp, d0, k - M_, phi, dphi);
            if (dim == 0) phi *= pr.q;
            wt[(p * 3 + dim) * 16 + k] = phi;
        }
        for (int p = tid; p < nb; p += NT) {
            int cx, cy, cz;
            unpack_cell(cell[start + b0 + p], cx, cy, cz);
            bs[p * 4 + 0] = cx - tx0; bs[p * 4 + 1] = cy - ty0; bs[p * 4 + 2] = cz - tz0;
        }
        __syncthreads();   // with double buffering this is the only barrier per batch
        if (tid < W * W) {
            for (int p = 0; p < nb; ++p) {
                const int bx = bs[p * 4], by = bs[p * 4 + 1], bz = bs[p * 4 + 2];
                const int oy = (ty - by + KW) % W, oz = (tz - bz + KW) % W;
                const T* wp_ = wt + p * 3 * 16;
                const T a = wp_[16 + oy] * wp_[32 + oz];
                T* row = tile_s + (bz + oz) * SPL + (by + oy) * SX + bx;
                T wx[16];
                if (sizeof(T) == 4) {
#pragma unroll
                    for (int v = 0; v < 4; ++v)
                        *reinterpret_cast<float4*>(&wx[4 * v]) = *reinterpret_cast<const float4*>(&wp_[4 * v]);
                } else {
#pragma unroll
                    for (int v = 0; v < 8; ++v)
                        *reinterpret_cast<double2*>(&wx[2 * v]) = *reinterpret_cast<const double2*>(&wp_[2 * v]);
                }
#pragma unroll
                for (int k = 0; k < W; ++k) row[k] += a * wx[k];
            }
        }
    }
    __syncthreads();
    // flush padded tile (origin = tile origin - m) to the periodic global grid
    for (int e = tid; e < TP * TP * TP; e += NT) {
        int lx = e % TP, t2 = e / TP, ly = t2 % TP, lz = t2 / TP;
        T v = tile_s[lz * SPL + ly * SX + lx];
        if (v != (T)0) {
            int gx = tx0 - M_ + lx, gy = ty0 - M_ + ly, gz = tz0 - M_ + lz;
            gx += gx < 0 ? g.n : 0; gx -= gx >= g.n ? g.n : 0;
            gy += gy < 0 ? g.n : 0; gy -= gy >= g.n ? g.n : 0;
            gz += gz < 0 ? g.n : 0; gz -= gz >= g.n ? g.n : 0;
            atomicAdd(&grid[((size_t)gz * g.n + gy) * g.n + gx], v);
        }
    }
}

// ------------------------------------------------------------------------ gather
template <typename T, int M_, int TILE>
constexpr size_t gather_smem_bytes() {
    using C = TileCfg<M_, TILE>;
    return sizeof(T) * ((size_t)C::CELLS + C::GATHER_WARPS * 6 * 16);
}

// kIk = false: analytic-derivative variant, F = pre*q * sum Psi[l] grad(phi phi phi)
//              with pre = -n/(pi L^2)  (exact gradient of the ENUF energy).
// kIk = true : one component d of the paper's ik variant, F[.,d] = pre*q * sum B_d[l] phi phi phi
//              with pre = 2/L^2 (Eq. 42).
template <typename T, int M_, int TILE, bool kIk>
__global__ void __launch_bounds__(TileCfg<M_, TILE>::GATHER_WARPS * 32)
gather_kernel(const T* __restrict__ field, const PRec<T>* __restrict__ rec,
              const uint32_t* __restrict__ cell, const uint32_t* __restrict__ idx,
              const uint32_t* __restrict__ offset, TileGeom g, WindowParams wp, T pre,
              int component, T* __restrict__ F) {
    using C = TileCfg<M_, TILE>;
    constexpr int W = C::W, TP = C::TP, SX = C::SX, SPL = C::SPL;
    constexpr int NT = C::GATHER_WARPS * 32;

    const int tile = blockIdx.x;
    const uint32_t start = offset[tile];
    const int cnt = (int)(offset[tile + 1] - start);
    if (cnt == 0) return;

    extern __shared__ __align__(16) unsigned char smem_raw[];
    T* tile_s = reinterpret_cast<T*>(smem_raw);
    T* wtab = tile_s + C::CELLS;    // [warps][6][16]: phi x,y,z then phi' x,y,z

    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int tx0 = (tile % g.nt) * TILE, ty0 = ((tile / g.nt) % g.nt) * TILE, tz0 = (tile / (g.nt * g.nt)) * TILE;

    for (int e = tid; e < TP * TP * TP; e += NT) {
        int lx = e % TP, t2 = e / TP, ly = t2 % TP, lz = t2 / TP;
        int gx = tx0 - M_ + lx, gy = ty0 - M_ + ly, gz = tz0 - M_ + lz;
        gx += gx < 0 ? g.n : 0; gx -= gx >= g.n ? g.n : 0;
        gy += gy < 0 ? g.n : 0; gy -= gy >= g.n ? g.n : 0;
        gz += gz < 0 ? g.n : 0; gz -= gz >= g.n ? g.n : 0;
        tile_s[lz * SPL + ly * SX + lx] = field[((size_t)gz * g.n + gy) * g.n + gx];
    }
    __syncthreads();

    T* wt = wtab + warp * 6 * 16;
    for (int p = warp; p < cnt; p += C::GATHER_WARPS) {
        const PRec<T> pr = rec[start + p];
        int cx, cy, cz;
        unpack_cell(cell[start + p], cx, cy, cz);
        const int bx = cx - tx0, by = cy - ty0, bz = cz - tz0;
        for (int e = lane; e < 3 * W; e += 32) {
            int dim = e / W, k = e - dim * W;
            T d0 = dim == 0 ? pr.dx : (dim == 1 ? pr.dy : pr.dz);
            T phi, dphi = (T)0;
            window_eval<T, !kIk>(wp, d0, k - M_, phi, dphi);
            wt[dim * 16 + k] = phi;
            if (!kIk) wt[(3 + dim) * 16 + k] = dphi;
        }
        __syncwarp();
        T wx[W], dwx[W];
#pragma unroll
        for (int k = 0; k < W; ++k) { wx[k] = wt[k]; if (!kIk) dwx[k] = wt[48 + k]; }
        T fx = (T)0, fy = (T)0, fz = (T)0;
        for (int rr = lane; rr < W * W; rr += 32) {
            const int rz = rr / W, ry = rr - rz * W;
            const T* row = tile_s + (bz + rz) * SPL + (by + ry) * SX + bx;
            T s0 = (T)0, s1 = (T)0;
#pragma unroll
            for (int k = 0; k < W; ++k) {
                T v = row[k];
                s0 += v * wx[k];
                if (!kIk) s1 += v * dwx[k];
            }
            const T wy = wt[16 + ry], wz = wt[32 + rz];
            if (kIk) {
                fx += s0 * (wy * wz);
            } else {
                const T dwy = wt[64 + ry], dwz = wt[80 + rz];
                fx += s1 * (wy * wz);
                fy += s0 * (dwy * wz);
                fz += s0 * (wy * dwz);
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
            const size_t j = idx[start + p];
            const T s = pre * pr.q;
            if (kIk) {
                F[3 * j + component] = s * fx;
            } else {
                F[3 * j] = s * fx; F[3 * j + 1] = s * fy; F[3 * j + 2] = s * fz;
            }
        }
        __syncwarp();
    }
}

}  // namespace enuf
