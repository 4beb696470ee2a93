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
    acc = __ffma2_rn(a, make_float2(w, w), acc);
}
__device__ __forceinline__ void fma_pair(double2& acc, const double2 a, const double w) {
    acc.x = fma(a.x, w, acc.x);
    acc.y = fma(a.y, w, acc.y);
}

// elementwise a + b and a * f on a pair (one packed instruction for fp32)
__device__ __forceinline__ float2 pair_add(const float2 a, const float2 b) { return __fadd2_rn(a, b); }
__device__ __forceinline__ double2 pair_add(double2 a, const double2 b) { a.x += b.x; a.y += b.y; return a; }
__device__ __forceinline__ float2 pair_scale(const float2 a, const float f) { return __fmul2_rn(a, make_float2(f, f)); }
__device__ __forceinline__ double2 pair_scale(double2 a, const double f) { a.x *= f; a.y *= f; return a; }

template <int M_>
struct SpreadCfg {
    static constexpr int W = 2 * M_ + 1;
    static constexpr int NT = 128;          // 4 warps: 2 x 2 patches of 8 x 8 cells
    static constexpr int CAP = NT;          // staged particles per chunk (one candidate per thread)
    // staged record of one particle: x row [16], y row [16], q * z row [16], (d0x, d0y, d0z, q).
    // Pitch 52 = 20 mod 32: the 16-byte stores of 8 consecutive slots cover all 32 banks.
    static constexpr int RP = 52, OX = 0, OY = 16, OZ = 32, OD = 48;
};

template <typename T, int M_>
constexpr size_t spread_smem_bytes() {
    using C = SpreadCfg<M_>;
    return sizeof(T) * (size_t)(C::CAP + 1) * C::RP + sizeof(int) * (size_t)C::CAP;
}

// kTrim (fp32 Kaiser-Bessel, m >= 5): particles are binned by the plane s = c_z - 1 + ks_z, ks = (d0 > 0),
// so that every particle of slab s has its 2m non-zero z weights on the planes s-m+1 .. s+m: the window
// is WZ = 2m planes, and the warps test their cells against the 2m-point x / y extents.
template <typename T, int M_, bool kTrim = false>
__global__ void __launch_bounds__(SpreadCfg<M_>::NT, sizeof(T) == 4 ? 7 : 2)
spread_kernel(const PSlot<T>* __restrict__ slots,
              const uint32_t* __restrict__ offset, TileGeom g, WindowParams wp,
              const __grid_constant__ PolyArg<M_> pa, int zchunk, T* __restrict__ grid) {
    using C = SpreadCfg<M_>;
    using P2 = typename Pair2<T>::type;
    constexpr int W = C::W, NT = C::NT, CAP = C::CAP, RP = C::RP, OX = C::OX, OY = C::OY, OZ = C::OZ, OD = C::OD;
    constexpr int WZ = W - (kTrim ? 1 : 0);            // planes in the register window
    constexpr int SLO = M_, SHI = kTrim ? M_ - 1 : M_;  // slabs z0 - SLO .. z1 - 1 + SHI reach the planes [z0, z1)

    extern __shared__ __align__(16) unsigned char smem_raw[];
    T* st = reinterpret_cast<T*>(smem_raw);            // [CAP + 1][RP] staged particle records; slot CAP is all zero
    int* sb = reinterpret_cast<int*>(st + (CAP + 1) * RP);   // [CAP] (bx + m) | (by + m) << 8 | ks_x << 16 | ks_y << 17
    __shared__ int rng_start[3][9], rng_cnt[3][9], rng_max[3];   // bin ranges of the slabs s - 1 / s / s + 1 / s + 2 (ring)
    __shared__ int nslot_s[2];                                   // staged count of the current / next round
    __shared__ unsigned char smask[CAP];                         // patch mask of a staged slot (copy of sb >> 20)
    // per warp: byte offsets (into st) of the staged particles that overlap the warp's cells, compacted
    __shared__ __align__(8) unsigned wlist[NT / 32][68];

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
            const int cnt = (int)(offset[nb_bin0 + cz + 1] - st);
            rng_start[buf][tid] = (int)st;
            rng_cnt[buf][tid] = cnt;
            const int mx = __reduce_max_sync(0x1ffu, cnt);       // lanes 0..8 of warp 0
            if (tid == 0) rng_max[buf] = mx;
        }
    };
    // cull mapping: kCullT threads per neighbouring column (9 x 14 = 126 of the 128 threads), thread
    // (cull_i, cull_k) tests the candidates cull_k, cull_k + 14, .. of column cull_i's bin -- no search for
    // the range a candidate belongs to
    constexpr int kCullT = NT / 9;
    const int cull_i = tid / kCullT < 9 ? tid / kCullT : -1, cull_k = tid % kCullT;
    const int cull_dx = (cull_i % 3 - 1) * kTile + M_, cull_dy = (cull_i / 3 - 1) * kTile + M_;
    const int s_begin = z0 - SLO, s_end = z1 + SHI;
    if (tid == 0) { nslot_s[0] = 0; nslot_s[1] = 0; }
    if (tid < RP) st[CAP * RP + tid] = (T)0;           // the padding record of odd-length visit lists
    load_ranges(s_begin, 0);
    if (s_begin + 1 < s_end) load_ranges(s_begin + 1, 1);
    __syncthreads();

    P2 acc[WZ];
#pragma unroll
    for (int k = 0; k < WZ; ++k) { acc[k].x = (T)0; acc[k].y = (T)0; }

    T* gout = grid + ((size_t)(Ty * kTile + ly)) * g.n + Tx * kTile + lx;
    const char* lane_xb = reinterpret_cast<const char*>(st + OX + lx);   // this lane's entries of slot 0's rows
    const char* lane_yb = reinterpret_cast<const char*>(st + OY + ly);
    const char* st_zb = reinterpret_cast<const char*>(st + OZ);

    // The kernel proceeds in rounds: one round = one chunk of candidates of one slab (a slab is a single round
    // unless a bin holds more than 2 kCullT particles or more than CAP were accepted):
    //   cull -> barrier -> window values -> barrier -> accumulate -> [slab done: store a plane, slide] -> cull of the
    //   NEXT round.  The cull only writes the packed positions sb[] and the raw records (words OD..OD+3 of a slot),
    //   which the accumulate phase does not read (it uses the rows and smask[]), so a warp that finishes its visits
    //   early culls the next round while the others are still accumulating: two barriers per round, and the
    //   cull's global-load latency overlaps the tail of the accumulate phase.
    int s = s_begin, rb = 0, c0 = 0, kk = 0, span = 2 * kCullT;
    {
        // cull the candidates [c0, c0 + span) of every bin against the column's halo: accepted ones are
        // staged (record + packed position) while slots last; returns nothing, the count is nslot_s
        auto cull = [&](int rbuf, int c0, int span, int kk) {
            const int my_start = cull_i >= 0 ? rng_start[rbuf][cull_i] : 0;
            const int my_cnt = cull_i >= 0 ? rng_cnt[rbuf][cull_i] : 0;
            // a thread has at most two candidates per chunk (span <= 2 kCullT): both cells are loaded before
            // either is examined, so the chunk costs one global-load latency, not two
            const int cend = min(my_cnt, c0 + span);
            const int ca = c0 + cull_k, cb = ca + kCullT;
            const uint32_t cell_a = ca < cend ? slots[my_start + ca].cell : 0u;
            const uint32_t cell_b = cb < cend ? slots[my_start + cb].cell : 0u;
            auto examine = [&](uint32_t pidx, uint32_t cellv) {
                int cx, cy, czp;
                unpack_cell(cellv, cx, cy, czp);
                const int bxm = (cx & (kTile - 1)) + cull_dx;   // bx + m, bx relative to the column
                const int bym = (cy & (kTile - 1)) + cull_dy;
                if ((unsigned)bxm < (unsigned)(kTile + 2 * M_) && (unsigned)bym < (unsigned)(kTile + 2 * M_)) {
                    const PRec<T> pr = slots[pidx].rec;
                    int pk = bxm | (bym << 8);
                    if (kTrim) pk |= (pr.dx > (T)0 ? 1 << 16 : 0) | (pr.dy > (T)0 ? 1 << 17 : 0);
                    // which of the four 8 x 8 warp patches the stencil touches (bits 20..23, warp order):
                    // it covers the column cells [b - (WZ-1), b], b = bxm (trimmed: bxm - 1 + ks)
                    const int bx2 = bxm + (kTrim ? (pr.dx > (T)0 ? 0 : -1) : 0);
                    const int by2 = bym + (kTrim ? (pr.dy > (T)0 ? 0 : -1) : 0);
                    const int ox = (bx2 >= 0 && bx2 - (WZ - 1) <= 7 ? 1 : 0) | (bx2 >= 8 && bx2 - (WZ - 1) <= 15 ? 2 : 0);
                    const int oy = (by2 >= 0 && by2 - (WZ - 1) <= 7 ? 1 : 0) | (by2 >= 8 && by2 - (WZ - 1) <= 15 ? 2 : 0);
                    const int mask = (oy & 1 ? ox : 0) | (oy & 2 ? ox << 2 : 0);
                    // a trimmed stencil at the far edge of the halo misses the column altogether: not staged
                    if (mask != 0) {
                        const int slot = atomicAdd(&nslot_s[kk], 1);
                        if (slot < CAP) {
                            *reinterpret_cast<PRec<T>*>(st + slot * RP + OD) = pr;
                            sb[slot] = pk | (mask << 20);
                        }
                    }
                }
            };
            if (ca < cend) examine((uint32_t)(my_start + ca), cell_a);
            if (cb < cend) examine((uint32_t)(my_start + cb), cell_b);
        };

        cull(rb, c0, span, kk);                                // round 0
        for (;;) {
            __syncthreads();                                   // this round's cull is complete; rows and smask are free
            int ns = nslot_s[kk];
            if (ns > CAP) {
                // more than CAP accepted (dense clusters): redo the chunk with one candidate per thread
                // (at most 9 * kCullT <= CAP accepted)
                __syncthreads();                 // every thread has read ns
                if (tid == 0) nslot_s[kk] = 0;
                __syncthreads();
                span = kCullT;
                cull(rb, c0, span, kk);
                __syncthreads();
                ns = nslot_s[kk];
            }
            if (tid == 0) nslot_s[kk ^ 1] = 0;                 // counter of the next round (nobody touches it now)
            if (c0 == 0 && s + 2 < s_end) load_ranges(s + 2, rb == 0 ? 2 : rb - 1);   // ring slot of slab s - 1
            // ---- window values: one task per (dimension, slot); dimension-major so warps stay uniform
            for (int t = tid; t < 3 * ns; t += NT) {
                const int dim = (t >= ns ? 1 : 0) + (t >= 2 * ns ? 1 : 0), slot = t - dim * ns;   // t < 3 ns
                T w[W], dw[W];
                const T d0 = st[slot * RP + OD + dim];
                stencil_weights<T, M_, false>(wp, pa, d0, w, dw);
                using V4 = typename Vec4<T>::type;
                if (dim == 2) {
                    smask[slot] = (unsigned char)((unsigned)sb[slot] >> 20);
                    const T q = st[slot * RP + OD + 3];
                    T r16[16];
#pragma unroll
                    for (int k = 0; k < 16; ++k)
                        r16[k] = k < WZ ? ((kTrim && d0 > (T)0) ? w[k + 1 < W ? k + 1 : 0] : w[k < W ? k : 0]) * q : (T)0;
                    V4* row4 = reinterpret_cast<V4*>(st + slot * RP + OZ);
#pragma unroll
                    for (int v = 0; v < 4; ++v) {
                        V4 o; o.x = r16[4 * v]; o.y = r16[4 * v + 1]; o.z = r16[4 * v + 2]; o.w = r16[4 * v + 3];
                        row4[v] = o;
                    }
                } else {
                    T* row = st + slot * RP + (dim == 0 ? OX : OY);
                    V4 z; z.x = (T)0; z.y = (T)0; z.z = (T)0; z.w = (T)0;
#pragma unroll
                    for (int v = 0; v < 4; ++v) reinterpret_cast<V4*>(row)[v] = z;
                    const int X0 = (dim == 0 ? (sb[slot] & 255) : ((sb[slot] >> 8) & 255)) - 2 * M_;   // cell of k = 0
#pragma unroll
                    for (int k = 0; k < W; ++k)
                        if ((unsigned)(X0 + k) < (unsigned)kTile) row[X0 + k] = w[k];
                }
            }
            __syncthreads();
            // ---- accumulate: each warp visits the staged particles that overlap its 8 x 8 cells
            for (int e0 = 0; e0 < ns; e0 += 64) {                      // 64 staged slots per pass
                // patch mask from the cull: does slot e0 + lane / e0 + 32 + lane touch this warp's cells?
                const bool ov0 = e0 + lane < ns && ((smask[e0 + lane] >> warp) & 1);
                const bool ov1 = e0 + 32 + lane < ns && ((smask[e0 + 32 + lane] >> warp) & 1);
                const unsigned om0 = __ballot_sync(0xffffffffu, ov0), om1 = __ballot_sync(0xffffffffu, ov1);
                const int cnt0 = __popc(om0), cnt = cnt0 + __popc(om1);
                if (cnt == 0) continue;
                // compact the overlapping slots into the warp's list (padded to an even length with the
                // zero record), then visit them two per trip: the loads of the second overlap the FMAs
                // of the first, and the trip has no data-dependent control flow
                unsigned* wl = wlist[warp];
                const unsigned below = (1u << lane) - 1u;
                if (ov0) wl[__popc(om0 & below)] = (unsigned)(e0 + lane) * (unsigned)(RP * sizeof(T));
                if (ov1) wl[cnt0 + __popc(om1 & below)] = (unsigned)(e0 + 32 + lane) * (unsigned)(RP * sizeof(T));
                if (lane == 0) wl[cnt] = (unsigned)CAP * (unsigned)(RP * sizeof(T));
                __syncwarp();
                uint2 oo = *reinterpret_cast<const uint2*>(wl);
                for (int i = 0; i < cnt; i += 2) {
                    const unsigned o1 = oo.x, o2 = oo.y;
                    oo = *reinterpret_cast<const uint2*>(wl + i + 2);        // next trip (list has 4 spare entries)
                    const P2 wx1 = *reinterpret_cast<const P2*>(lane_xb + o1);
                    const T wy1 = *reinterpret_cast<const T*>(lane_yb + o1);
                    const P2 wx2 = *reinterpret_cast<const P2*>(lane_xb + o2);
                    const T wy2 = *reinterpret_cast<const T*>(lane_yb + o2);
                    const P2 a1 = pair_scale(wx1, wy1), a2 = pair_scale(wx2, wy2);
                    // q * z rows: 16-byte vector loads (slot pitch and OZ are multiples of 16 bytes)
                    using V4 = typename Vec4<T>::type;
                    constexpr int NV = (WZ + 3) / 4;
                    V4 z1[NV], z2[NV];
#pragma unroll
                    for (int v = 0; v < NV; ++v) z1[v] = reinterpret_cast<const V4*>(st_zb + o1)[v];
#pragma unroll
                    for (int v = 0; v < NV; ++v) z2[v] = reinterpret_cast<const V4*>(st_zb + o2)[v];
                    const T* wz1 = reinterpret_cast<const T*>(z1);
                    const T* wz2 = reinterpret_cast<const T*>(z2);
#pragma unroll
                    for (int k = 0; k < WZ; ++k) fma_pair(acc[k], a1, wz1[k]);
#pragma unroll
                    for (int k = 0; k < WZ; ++k) fma_pair(acc[k], a2, wz2[k]);
                }
                __syncwarp();                    // the list is rewritten by the next group of 64 slots
            }
            // ---- next round: the rest of this slab, or the next slab after storing the finished plane
            c0 += span;
            span = 2 * kCullT;
            if (c0 >= rng_max[rb]) {
                // the lowest plane of the window (s - m, trimmed: s - m + 1) is complete: store it, slide
                const int zo = s - SHI;
                if (zo >= z0) *reinterpret_cast<P2*>(gout + (size_t)zo * g.n * g.n) = acc[0];
#pragma unroll
                for (int k = 0; k + 1 < WZ; ++k) acc[k] = acc[k + 1];
                acc[WZ - 1].x = (T)0; acc[WZ - 1].y = (T)0;
                ++s; rb = rb == 2 ? 0 : rb + 1; c0 = 0;
                if (s >= s_end) break;
            }
            kk ^= 1;
            cull(rb, c0, span, kk);                            // no barrier: see the comment above the loop
        }
    }
}

}  // namespace enuf
