// Step a1 -- wrap positions (x = r/L; R10) and counting-sort the charged
// particles by grid tile: histogram -> exclusive scan -> scatter.  The cell index c and
// the fractional offset d0 = u - c are formed in fp64 in the order
//   x = r/L;  x -= floor(x);  u = n*x;  c = floor(u + 1/2)
// for both precisions (an fp32 u would lose the offset: ulp(256) ~ 1.5e-5 cells), so the
// binned record carries d0 to full precision of T.
#pragma once

#include "enuf_common.cuh"

namespace enuf {

struct CellOfParticle {
    int c[3];        // nearest grid point per dimension, wrapped into [0, n)
    double d0[3];    // u - (unwrapped c), in [-1/2, 1/2]
};

template <typename T>
__device__ __forceinline__ CellOfParticle locate(const T* __restrict__ r, int64_t j, double L, int n) {
    CellOfParticle o;
#pragma unroll
    for (int t = 0; t < 3; ++t) {
        double x = __ddiv_rn((double)r[3 * j + t], L);
        x -= floor(x);
        if (x >= 1.0) x = 0.0;
        double u = __dmul_rn((double)n, x);
        double c = floor(__dadd_rn(u, 0.5));
        o.d0[t] = u - c;
        int ci = (int)c;
        o.c[t] = ci >= n ? ci - n : ci;
    }
    return o;
}

__device__ __forceinline__ int tile_of(const int c[3], const TileGeom& g) {
    int tx = c[0] / g.T, ty = c[1] / g.T, tz = c[2] / g.T;
    return (tz * g.nt + ty) * g.nt + tx;
}

// Histogram of charged particles per tile; neutral particles get F = 0 here and are dropped.
template <typename T>
__global__ void __launch_bounds__(256)
bin_count_kernel(const T* __restrict__ r, const T* __restrict__ q, T* __restrict__ F, int64_t N,
                 double L, TileGeom g, uint32_t* __restrict__ count) {
    int64_t j = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (j >= N) return;
    if (q[j] == (T)0) {
        F[3 * j] = (T)0; F[3 * j + 1] = (T)0; F[3 * j + 2] = (T)0;
        return;
    }
    CellOfParticle p = locate(r, j, L, g.n);
    atomicAdd(&count[tile_of(p.c, g)], 1u);
}

// Exclusive scan of count[0..ntiles) into offset[0..ntiles]; zeroes cursor. One CTA.
static __global__ void __launch_bounds__(1024)
bin_scan_kernel(const uint32_t* __restrict__ count, uint32_t* __restrict__ offset,
                uint32_t* __restrict__ cursor, int ntiles) {
    __shared__ uint32_t warp_sums[32];
    __shared__ uint32_t carry_s;
    const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
    if (threadIdx.x == 0) carry_s = 0;
    __syncthreads();
    for (int base = 0; base < ntiles; base += 1024) {
        int i = base + threadIdx.x;
        uint32_t v = i < ntiles ? count[i] : 0u;
        uint32_t inc = v;
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) {
            uint32_t t = __shfl_up_sync(0xffffffffu, inc, o);
            if (lane >= o) inc += t;
        }
        if (lane == 31) warp_sums[wid] = inc;
        __syncthreads();
        if (wid == 0) {
            uint32_t ws = warp_sums[lane], winc = ws;
#pragma unroll
            for (int o = 1; o < 32; o <<= 1) {
                uint32_t t = __shfl_up_sync(0xffffffffu, winc, o);
                if (lane >= o) winc += t;
            }
            warp_sums[lane] = winc - ws;   // exclusive prefix of warp totals
        }
        __syncthreads();
        uint32_t carry = carry_s;
        uint32_t excl = carry + warp_sums[wid] + inc - v;
        if (i < ntiles) { offset[i] = excl; cursor[i] = 0u; }
        __syncthreads();
        if (threadIdx.x == 1023) carry_s = excl + v;
        __syncthreads();
    }
    if (threadIdx.x == 0) offset[ntiles] = carry_s;
}

// Scatter into tile order.  The order inside a tile follows the atomic cursor (any order is
// a valid sort; sums downstream differ only in rounding order, R22).
template <typename T>
__global__ void __launch_bounds__(256)
bin_scatter_kernel(const T* __restrict__ r, const T* __restrict__ q, int64_t N, double L, TileGeom g,
                   const uint32_t* __restrict__ offset, uint32_t* __restrict__ cursor,
                   PRec<T>* __restrict__ rec, uint32_t* __restrict__ cell, uint32_t* __restrict__ idx) {
    int64_t j = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (j >= N) return;
    T qj = q[j];
    if (qj == (T)0) return;
    CellOfParticle p = locate(r, j, L, g.n);
    int t = tile_of(p.c, g);
    uint32_t pos = offset[t] + atomicAdd(&cursor[t], 1u);
    PRec<T> o;
    o.dx = (T)p.d0[0]; o.dy = (T)p.d0[1]; o.dz = (T)p.d0[2]; o.q = qj;
    rec[pos] = o;
    cell[pos] = pack_cell(p.c[0], p.c[1], p.c[2]);
    idx[pos] = (uint32_t)j;
}

}  // namespace enuf
