// Step a2 -- spreading (adjoint NFFT, part 1):
//   g[l] = sum_j q_j phi(u_jx - l_x) phi(u_jy - l_y) phi(u_jz - l_z), l periodic.
//
// Output-stationary, sliding z-window.  A CTA owns a 16 x 16 column of grid cells in
// (x, y) and a chunk [z0, z1) of grid planes.  Every lane owns two x-adjacent cells of the
// column and keeps, in registers, the partial sums of those two cells on the W = 2m+1
// consecutive planes z = s-m .. s+m that the particles of slab s (nearest plane c_z = s)
// can reach.  The CTA walks s upwards: after slab s, plane s-m is complete, is written to
// the grid with one plain coalesced store, and the window slides by one plane.  So
//   - every grid value is written exactly once: no atomics, no clearing of the grid,
//     and the sum for a cell is formed in registers (no shared-memory read-modify-write);
//   - per (warp, particle) visit the work is W packed FMAs acc[k] += (a0, a1) * wz[k],
//     with a0, a1 = wx[cell] * wy[cell] read from zero-padded per-particle rows.
// The particles of slab s that reach the column come from the 3 x 3 neighbouring columns'
// bins (TileGeom); they are culled against the column's halo of m cells, their 3 W window
// values are computed once per CTA (the paper's "window values computed in local memory",
// PAPER.md:519) and staged in shared memory; each of the four warps (8 x 8 cells) then
// visits only the particles whose stencil overlaps its cells.
#pragma once

#include "enuf_common.cuh"

namespace enuf {

template <typename T> struct Pair2;
template <> struct Pair2<float> { using type = float2; };
template <> struct Pair2<double> { using type = double2; };

// acc += a * w (both halves), one FFMA2 for fp32 on sm_100a
__device__ __forceinline__ void fma_pair(float2& acc, const float2 a, const float w) {
    unsigned long long A, C, Wv;
    const float2 w2 = make_float2(w, w);
    A = *reinterpret_cast<const unsigned long long*>(&a);
    C = *reinterpret_cast<unsigned long long*>(&acc);
    Wv = *reinterpret_cast<const unsigned long long*>(&w2);
    asm("fma.rn.f32x2 %0, %1, %2, %0;" : "+l"(C) : "l"(A), "l"(Wv));
    acc = *reinterpret_cast<float2*>(&C);
}
__device__ __forceinline__ void fma_pair(double2& acc, const double2 a, const double w) {
    acc.x = fma(a.x, w, acc.x);
    acc.y = fma(a.y, w, acc.y);
}

template <int M_>
struct SpreadCfg {
    static constexpr int W = 2 * M_ + 1;
    static constexpr int NT = 128;          // 4 warps: 2 x 2 patches of 8 x 8 cells
    static constexpr int CAP = NT;          // staged particles per chunk (one candidate per thread)
    static constexpr int ROW = 16;          // row length of the staged x / y / z weight rows
};

template <typename T, int M_>
constexpr size_t spread_smem_bytes() {
    using C = SpreadCfg<M_>;
    return sizeof(T) * (size_t)C::CAP * (3 * C::ROW + 4) + sizeof(int) * (size_t)C::CAP;
}

template <typename T, int M_>
__global__ void __launch_bounds__(SpreadCfg<M_>::NT)
spread_kernel(const PRec<T>* __restrict__ rec, const uint32_t* __restrict__ cell,
              const uint32_t* __restrict__ offset, TileGeom g, WindowParams wp,
              const __grid_constant__ PolyArg<M_> pa, int zchunk, T* __restrict__ grid) {
    using C = SpreadCfg<M_>;
    using P2 = typename Pair2<T>::type;
    constexpr int W = C::W, NT = C::NT, CAP = C::CAP, ROW = C::ROW;

    extern __shared__ __align__(16) unsigned char smem_raw[];
    T* wxr = reinterpret_cast<T*>(smem_raw);          // [CAP][ROW] x weights on the column's 16 cells
    T* wyr = wxr + CAP * ROW;                          // [CAP][ROW]
    T* wzr = wyr + CAP * ROW;                          // [CAP][ROW] q * z weights, k = 0..W-1
    T* sd = wzr + CAP * ROW;                           // [CAP][4]   d0x, d0y, d0z, q
    int* sb = reinterpret_cast<int*>(sd + CAP * 4);    // [CAP]      (bx + m) | (by + m) << 8
    __shared__ int rng_start[2][9], rng_cnt[2][9];
    __shared__ int nslot_s;

    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int Tx = blockIdx.x % g.nt, Ty = blockIdx.x / g.nt;
    const int z0 = blockIdx.y * zchunk, z1 = min(g.n, z0 + zchunk);
    const int px = (warp & 1) * 8, py = (warp >> 1) * 8;           // warp patch origin in the column
    const int lx = px + (lane & 3) * 2, ly = py + (lane >> 2);     // this lane's two cells: (lx, ly), (lx+1, ly)

    // the 9 neighbouring columns (tid < 9): bin of plane 0
    int nb_bin0 = 0;
    if (tid < 9) {
        int ty = Ty + tid / 3 - 1, tx = Tx + tid % 3 - 1;
        ty += ty < 0 ? g.nt : 0; ty -= ty >= g.nt ? g.nt : 0;
        tx += tx < 0 ? g.nt : 0; tx -= tx >= g.nt ? g.nt : 0;
        nb_bin0 = (ty * g.nt + tx) * g.n;
    }
    auto load_ranges = [&](int s, int buf) {
        if (tid < 9) {
            const int cz = s < 0 ? s + g.n : (s >= g.n ? s - g.n : s);
            const uint32_t st = offset[nb_bin0 + cz];
            rng_start[buf][tid] = (int)st;
            rng_cnt[buf][tid] = (int)(offset[nb_bin0 + cz + 1] - st);
        }
    };
    if (tid == 0) nslot_s = 0;
    load_ranges(z0 - M_, 0);

    P2 acc[W];
#pragma unroll
    for (int k = 0; k < W; ++k) { acc[k].x = (T)0; acc[k].y = (T)0; }

    T* gout = grid + ((size_t)(Ty * kTile + ly)) * g.n + Tx * kTile + lx;

    int buf = 0;
    for (int s = z0 - M_; s < z1 + M_; ++s, buf ^= 1) {
        __syncthreads();      // ranges of slab s visible; all warps are done with the previous slab
        if (s + 1 < z1 + M_) load_ranges(s + 1, buf ^ 1);
        int pref[10];
        pref[0] = 0;
#pragma unroll
        for (int i = 0; i < 9; ++i) pref[i + 1] = pref[i] + rng_cnt[buf][i];
        const int total = pref[9];

        for (int c0 = 0; c0 < total; c0 += NT) {
            // ---- cull: one candidate per thread
            const int c = c0 + tid;
            bool take = false;
            int bxm = 0, bym = 0;
            uint32_t pidx = 0;
            if (c < total) {
                int i = 0;
#pragma unroll
                for (int e = 1; e < 9; ++e) i += (c >= pref[e]) ? 1 : 0;
                int pb = 0;
#pragma unroll
                for (int e = 1; e < 9; ++e) pb = (i == e) ? pref[e] : pb;
                pidx = (uint32_t)(rng_start[buf][i] + (c - pb));
                int cx, cy, czp;
                unpack_cell(cell[pidx], cx, cy, czp);
                bxm = (cx & (kTile - 1)) + (i % 3 - 1) * kTile + M_;      // bx + m, bx relative to the column
                bym = (cy & (kTile - 1)) + (i / 3 - 1) * kTile + M_;
                take = (unsigned)bxm < (unsigned)(kTile + 2 * M_) && (unsigned)bym < (unsigned)(kTile + 2 * M_);
            }
            const unsigned tmask = __ballot_sync(0xffffffffu, take);
            if (tmask) {
                int base = 0;
                if (lane == 0) base = atomicAdd(&nslot_s, __popc(tmask));
                base = __shfl_sync(0xffffffffu, base, 0);
                if (take) {
                    const int slot = base + __popc(tmask & ((1u << lane) - 1u));
                    const PRec<T> pr = rec[pidx];
                    sd[slot * 4 + 0] = pr.dx; sd[slot * 4 + 1] = pr.dy; sd[slot * 4 + 2] = pr.dz; sd[slot * 4 + 3] = pr.q;
                    sb[slot] = bxm | (bym << 8);
                }
            }
            __syncthreads();
            const int ns = nslot_s;
            // ---- window values: one task per (dimension, slot); dimension-major so warps stay uniform
            for (int t = tid; t < 3 * ns; t += NT) {
                const int dim = t / ns, slot = t - dim * ns;
                T w[W], dw[W];
                stencil_weights<T, M_, false>(wp, pa, sd[slot * 4 + dim], w, dw);
                if (dim == 2) {
                    const T q = sd[slot * 4 + 3];
#pragma unroll
                    for (int k = 0; k < W; ++k) wzr[slot * ROW + k] = w[k] * q;
                } else {
                    T* row = (dim == 0 ? wxr : wyr) + slot * ROW;
#pragma unroll
                    for (int e = 0; e < ROW; ++e) row[e] = (T)0;
                    const int X0 = (dim == 0 ? (sb[slot] & 255) : (sb[slot] >> 8)) - 2 * M_;   // cell of k = 0
#pragma unroll
                    for (int k = 0; k < W; ++k)
                        if ((unsigned)(X0 + k) < (unsigned)kTile) row[X0 + k] = w[k];
                }
            }
            __syncthreads();
            if (tid == 0) nslot_s = 0;      // every thread has read ns; the next cull starts after a barrier
            // ---- accumulate: each warp visits the staged particles that overlap its 8 x 8 cells
            for (int e0 = 0; e0 < ns; e0 += 32) {
                bool ov = false;
                if (e0 + lane < ns) {
                    const int v = sb[e0 + lane];
                    const int bx2 = v & 255, by2 = v >> 8;            // stencil covers [b - 2m, b] in column cells
                    ov = bx2 >= px && bx2 - 2 * M_ <= px + 7 && by2 >= py && by2 - 2 * M_ <= py + 7;
                }
                unsigned om = __ballot_sync(0xffffffffu, ov);
                while (om) {
                    const int e = e0 + __ffs(om) - 1;
                    om &= om - 1;
                    const P2 wx2 = *reinterpret_cast<const P2*>(&wxr[e * ROW + lx]);
                    const T wy = wyr[e * ROW + ly];
                    P2 a; a.x = wx2.x * wy; a.y = wx2.y * wy;
                    const T* wz = &wzr[e * ROW];
#pragma unroll
                    for (int k = 0; k < W; ++k) fma_pair(acc[k], a, wz[k]);
                }
            }
            if (c0 + NT < total) __syncthreads();     // staging buffers are reused by the next chunk
        }
        // ---- plane z = s - m is complete: store it and slide the window
        const int zo = s - M_;
        if (zo >= z0) *reinterpret_cast<P2*>(gout + (size_t)zo * g.n * g.n) = acc[0];
#pragma unroll
        for (int k = 0; k + 1 < W; ++k) acc[k] = acc[k + 1];
        acc[W - 1].x = (T)0; acc[W - 1].y = (T)0;
    }
}

}  // namespace enuf
