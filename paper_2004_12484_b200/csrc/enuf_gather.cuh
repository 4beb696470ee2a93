// Step a6 -- interpolating (forward NFFT, last part; Eq. 42 :340).
//
// One CTA per 16^3 grid tile, working on the tile's particles (16 ranges of the sorted array, one
// per plane; TileGeom), with the tile plus a halo of m cells per side ((16+2m)^3 values) held in
// shared memory (staged with cp.async).  Every warp takes a contiguous share of the tile's
// particles (shares differ by at most one), five at a time: first the 3 W window values and derivatives of those particles are computed once
// (one lane per particle and dimension) and kept on chip, then the warp
// contracts the (2m+1)^3 stencil of one particle after the other: every lane owns x-rows of
// the stencil (row strides chosen so that the 32 rows a warp reads at once fall in 32
// different banks), forms s = sum_x Psi (phi, phi') with
// packed FMAs, and the three force components come out of one pass over the field
// ("forces in 3D packed into a single calculation entity").
#pragma once

#include <type_traits>

#include "enuf_common.cuh"
#include "enuf_spread.cuh"   // Pair2, fma_pair

namespace enuf {

// (row stride, plane stride) of the shared tile, found by search: the 32 stencil rows (rz, ry) =
// divmod(lane + 32 it, WE) a warp reads at once fall in 32 different banks.  kTrim: WE = 2m.
template <int M_, bool kTrim> struct GatherStride;
template <> struct GatherStride<1, false> { static constexpr int SX = 18, SPL = 325; };
template <> struct GatherStride<2, false> { static constexpr int SX = 21, SPL = 425; };
template <> struct GatherStride<3, false> { static constexpr int SX = 23, SPL = 513; };
template <> struct GatherStride<4, false> { static constexpr int SX = 25, SPL = 609; };
template <> struct GatherStride<5, false> { static constexpr int SX = 27, SPL = 713; };
template <> struct GatherStride<6, false> { static constexpr int SX = 29, SPL = 825; };
// Trimmed fp32 plans read the stencil rows with 8-byte loads (kPair below): even row stride, and a plane
// stride = 8 (m = 6) / 12 (m = 5) mod 32 so that the 16 rows x 2 words of each half-warp hit 32 different banks.
template <> struct GatherStride<5, true> { static constexpr int SX = 30, SPL = 26 * 30; };
template <> struct GatherStride<6, true> { static constexpr int SX = 30, SPL = 28 * 30; };

// kTrim (fp32 Kaiser-Bessel, m >= 5; enuf_common.cuh): the window vanishes beyond |d| = m, so of the
// 2m+1 stencil points per dimension the outermost one on the far side of the particle carries an exact
// zero.  The kernels then work on the WE = 2m points [c - m + ks, c + m - 1 + ks], ks = (d0 > 0).
template <int M_, bool kTrim = false>
struct GatherCfg {
    static constexpr int W = 2 * M_ + 1;
    static constexpr int WE = W - (kTrim ? 1 : 0);              // stencil points per dimension actually visited
    static constexpr int TP = kTile + 2 * M_;                   // padded tile edge
    // kPair: the x rows of the shared tile start on an even grid column (halo XS = m rounded up to even) so
    // that staging copies and stencil-row loads move aligned pairs (Psi[x], Psi[x+1])
    static constexpr bool kPair = kTrim;
    static constexpr int XS = kPair ? ((M_ + 1) & ~1) : M_;     // x halo on the low side
    static constexpr int TPX = kTile + 2 * XS;                  // staged row length
    static constexpr int SX = GatherStride<M_, kTrim>::SX;
    static constexpr int SPL = GatherStride<M_, kTrim>::SPL;
    static constexpr int CELLS = ((TP * SPL + 3) / 4) * 4;      // shared tile size in elements (16 B multiple)
    static constexpr int WARPS = 12;
    static constexpr int NT = WARPS * 32;
    // kPairWarp (trimmed stencils of 4 k points, i.e. fp32 Kaiser-Bessel m = 6): a warp contracts TWO particles at a
    // time, 16 lanes each; a lane owns the (WE/4)^2 rows (y, z) = (ya + 4 i, zb + 4 j) of the stencil and keeps their
    // y and z weights in registers
    static constexpr bool kPairWarp = kPair && WE % 4 == 0;
    static constexpr int PBW = kPairWarp ? 4 : 5;               // particles per warp batch (3 lanes per particle compute weights); shared memory: 2 CTAs per SM
    static constexpr int ITER = (WE * WE + 31) / 32;            // stencil rows per lane
    static constexpr int WP = 14;                               // pitch of a (phi, phi') weight row: >= WE, 16-byte aligned; 28 words: the
                                                                //   12 lanes that store a batch's rows 16 bytes at a time collide two-way, not three-way
    static constexpr int PERM = 64;                             // kPairWarp: particles a warp sorts by row parity at a time
};

template <typename T, int M_, bool kTrim = false>
constexpr size_t gather_smem_bytes() {
    using C = GatherCfg<M_, kTrim>;
    // tile + per warp and batch particle: (phi, phi') pairs [3][WP], pre*q, tile offset, caller index
    return sizeof(T) * ((size_t)C::CELLS + (size_t)C::WARPS * C::PBW * (3 * C::WP * 2 + 1))
           + sizeof(int) * 2 * C::WARPS * C::PBW + (C::kPairWarp ? sizeof(uint32_t) * C::WARPS * C::PERM : 0);
}

__device__ __forceinline__ void cp_async_4(void* smem_dst, const void* gmem_src) {
    const unsigned d = (unsigned)__cvta_generic_to_shared(smem_dst);
    asm volatile("cp.async.ca.shared.global [%0], [%1], 4;" ::"r"(d), "l"(gmem_src) : "memory");
}
__device__ __forceinline__ void cp_async_8(void* smem_dst, const void* gmem_src) {
    const unsigned d = (unsigned)__cvta_generic_to_shared(smem_dst);
    asm volatile("cp.async.ca.shared.global [%0], [%1], 8;" ::"r"(d), "l"(gmem_src) : "memory");
}
__device__ __forceinline__ void cp_async_wait_all() { asm volatile("cp.async.wait_all;" ::: "memory"); }

// kIk = false: analytic-derivative variant, F = pre*q * sum Psi[l] grad(phi phi phi)
//              with pre = -n/(pi L^2)  (exact gradient of the ENUF energy).
// kIk = true : one component d of the paper's ik variant, F[.,d] = pre*q * sum B_d[l] phi phi phi
//              with pre = 2/L^2 (Eq. 42).
template <typename T, int M_, bool kIk, bool kTrim = false>
__global__ void __launch_bounds__((GatherCfg<M_, kTrim>::NT), (sizeof(T) == 4 ? 2 : 1))
gather_kernel(const T* __restrict__ field, const PSlot<T>* __restrict__ slots,
              const uint32_t* __restrict__ offset, TileGeom g, WindowParams wp,
              const __grid_constant__ PolyArg<M_> pa, T pre, int component, T* __restrict__ F, T ry, T rz) {
    pdl_prologue();
    using C = GatherCfg<M_, kTrim>;
    using P2 = typename Pair2<T>::type;
    constexpr int W = C::W, WE = C::WE, TP = C::TP, SX = C::SX, SPL = C::SPL, PBW = C::PBW, ITER = C::ITER, WP = C::WP;

    // tile (Tx, Ty, Tz): the particles of its 16 planes are 16 ranges of the sorted array, bins
    // bin_index(Tx, Ty, 16 Tz + zl) (TileGeom); pre_s[zl] = particles of the planes before zl
    const int ntz = g.n / kTile;
    const int Tz = blockIdx.x % ntz, col = blockIdx.x / ntz;
    const int Tx = col % g.nt, Ty = col / g.nt;
    __shared__ uint32_t st_s[kTile];
    __shared__ int pre_s[kTile + 1];
    if (threadIdx.x < 32) {
        const int zl = threadIdx.x & (kTile - 1);
        const int b = bin_index(g, Tx, Ty, Tz * kTile + zl);
        const uint32_t st = offset[b];
        int c = (int)(offset[b + 1] - st), inc = c;
#pragma unroll
        for (int o = 1; o < kTile; o <<= 1) {
            const int t = __shfl_up_sync(0xffffffffu, inc, o, kTile);
            if (zl >= o) inc += t;
        }
        if (threadIdx.x < kTile) {
            st_s[zl] = st; pre_s[zl] = inc - c;
            if (zl == kTile - 1) pre_s[kTile] = inc;
        }
    }
    __syncthreads();
    const int cnt = pre_s[kTile];
    if (cnt == 0) return;
    // sorted-array index of the tile's p-th particle
    auto slot_of = [&](int p) -> uint32_t {
        int lo = 0;
        if (pre_s[lo + 8] <= p) lo += 8;
        if (pre_s[lo + 4] <= p) lo += 4;
        if (pre_s[lo + 2] <= p) lo += 2;
        if (pre_s[lo + 1] <= p) lo += 1;
        return st_s[lo] + (uint32_t)(p - pre_s[lo]);
    };

    extern __shared__ __align__(16) unsigned char smem_raw[];
    T* tile_s = reinterpret_cast<T*>(smem_raw);
    P2* wtab_all = reinterpret_cast<P2*>(tile_s + C::CELLS);            // [WARPS][PBW][3][WP] (phi, phi')
    T* q_all = reinterpret_cast<T*>(wtab_all + C::WARPS * PBW * 3 * WP); // [WARPS][PBW] pre * q
    int* base_all = reinterpret_cast<int*>(q_all + C::WARPS * PBW);     // [WARPS][PBW] tile offset of the stencil origin
    int* idx_all = base_all + C::WARPS * PBW;                           // [WARPS][PBW] caller index

    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int tx0 = Tx * kTile, ty0 = Ty * kTile, tz0 = Tz * kTile;

    // ---- stage the padded tile asynchronously
    if constexpr (C::kPair && sizeof(T) == 4) {
        // 8-byte copies: a warp takes whole planes (lz = warp, warp + WARPS, ..), each half-warp moving one
        // row of TPX / 2 pairs per step
        constexpr int PAIRS = C::TPX / 2;
        const int half = lane >> 4, pxi = lane & 15;
        int gx = tx0 - C::XS + 2 * pxi;
        gx += gx < 0 ? g.n : 0; gx -= gx >= g.n ? g.n : 0;
        int gy0 = ty0 - M_ + half;
        gy0 += gy0 < 0 ? g.n : 0;
        const size_t nn = (size_t)g.n;
        if (pxi < PAIRS) {
            for (int lz = warp; lz < TP; lz += C::WARPS) {
                int gz = tz0 - M_ + lz;
                gz += gz < 0 ? g.n : 0; gz -= gz >= g.n ? g.n : 0;
                const T* src = field + (size_t)gz * nn * nn + gx;
                T* dst = tile_s + lz * SPL + half * SX + 2 * pxi;
                int gy = gy0;
#pragma unroll
                for (int j = 0; j < (TP + 1) / 2; ++j) {
                    if (2 * j + 1 < TP || half == 0) cp_async_8(dst + 2 * j * SX, src + (size_t)gy * nn);
                    gy += 2; gy -= gy >= g.n ? g.n : 0;
                }
            }
        }
    } else {
        int gx = tx0 - M_ + lane;
        gx += gx < 0 ? g.n : 0; gx -= gx >= g.n ? g.n : 0;
        for (int lz = 0; lz < TP; ++lz) {
            int gz = tz0 - M_ + lz;
            gz += gz < 0 ? g.n : 0; gz -= gz >= g.n ? g.n : 0;
            const T* plane = field + (size_t)gz * g.n * g.n + gx;
            T* dst = tile_s + lz * SPL + lane;
#pragma unroll
            for (int r = 0; r < (TP + C::WARPS - 1) / C::WARPS; ++r) {
                const int ly = warp + r * C::WARPS;
                int gy = ty0 - M_ + ly;
                gy += gy < 0 ? g.n : 0; gy -= gy >= g.n ? g.n : 0;
                if (ly < TP && lane < TP) {
                    if (sizeof(T) == 4) cp_async_4(dst + ly * SX, plane + (size_t)gy * g.n);
                    else cp_async_8(dst + ly * SX, plane + (size_t)gy * g.n);
                }
            }
        }
    }

    if constexpr (C::kPairWarp && sizeof(T) == 4) {
        // ================================================= two particles per warp (header of GatherCfg)
        constexpr int NR = WE / 4;                               // rows per lane and direction
        uint32_t* perm = reinterpret_cast<uint32_t*>(idx_all + C::WARPS * PBW) + warp * C::PERM;
        P2* wtab = wtab_all + warp * PBW * 3 * WP;
        T* q_s = q_all + warp * PBW;
        int* base_s = base_all + warp * PBW;
        int* idx_s = idx_all + warp * PBW;
        const int half = lane >> 4, l16 = lane & 15, ya = l16 & 3, zb = l16 >> 2;
        const int rowbase = zb * SPL + ya * SX;                  // row (i, j) of the lane: + 4 i SX + 4 j SPL
        const unsigned below = (1u << lane) - 1u;
        const int share = cnt / C::WARPS, extra = cnt - share * C::WARPS;
        const int wbeg = warp * share + min(warp, extra), wend = wbeg + share + (warp < extra ? 1 : 0);
        bool tile_ready = false;
        for (int c0 = wbeg; c0 < wend; c0 += C::PERM) {
            const int n = min(C::PERM, wend - c0);
            // ---- particles whose stencil rows start on an even tile column first, the odd ones after: the two
            //      particles of a pair then take the same (aligned / unaligned) row-load path, except one pair per chunk
            if (n <= 2) {
                // one pair: nothing to sort (and no global-load round trip for the cell words)
                if (lane < n) perm[lane] = slot_of(c0 + lane);
                __syncwarp();
            } else {
                uint32_t gi[2]; bool ev[2], od[2];
#pragma unroll
                for (int h = 0; h < 2; ++h) {
                    const int pl = 32 * h + lane;
                    gi[h] = 0; ev[h] = od[h] = false;
                    if (pl < n) {
                        gi[h] = slot_of(c0 + pl);
                        const uint32_t cw = slots[gi[h]].cell;
                        const bool odd = (((cw & 1023u) + ((cw >> 30) & 1u) + (unsigned)(C::XS - M_)) & 1u) != 0u;
                        ev[h] = !odd; od[h] = odd;
                    }
                }
                const unsigned e0 = __ballot_sync(0xffffffffu, ev[0]), e1 = __ballot_sync(0xffffffffu, ev[1]);
                const unsigned o0 = __ballot_sync(0xffffffffu, od[0]), o1 = __ballot_sync(0xffffffffu, od[1]);
                const int ne = __popc(e0) + __popc(e1);
                __syncwarp();
                if (ev[0]) perm[__popc(e0 & below)] = gi[0];
                if (ev[1]) perm[__popc(e0) + __popc(e1 & below)] = gi[1];
                if (od[0]) perm[ne + __popc(o0 & below)] = gi[0];
                if (od[1]) perm[ne + __popc(o0) + __popc(o1 & below)] = gi[1];
                __syncwarp();
            }
            for (int b0 = 0; b0 < n; b0 += PBW) {
                const int nb = min(PBW, n - b0);
                // ---- window values of the batch: one lane per (dimension, particle)
                if (lane < 3 * nb) {
                    const int dim = lane / nb, slot = lane - dim * nb;
                    const uint32_t gi = perm[b0 + slot];
                    const PSlot<T> sl = slots[gi];
                    const PRec<T> pr = sl.rec;
                    const T d0 = dim == 0 ? pr.dx : (dim == 1 ? pr.dy : pr.dz);
                    T w[W], dw[W];
                    stencil_weights<T, M_, !kIk, true>(wp, pa, d0, w, dw);   // packed Horner chains
                    P2* row = wtab + (slot * 3 + dim) * WP;
                    const bool sh = d0 > (T)0;                  // ks = 1: the k = 0 point is the zero one
#pragma unroll
                    for (int k = 0; k < WE; k += 2) {
                        typename Vec4<T>::type v4;
                        v4.x = sh ? w[k + 1] : w[k];      v4.y = sh ? dw[k + 1] : dw[k];
                        v4.z = sh ? w[k + 2] : w[k + 1];  v4.w = sh ? dw[k + 2] : dw[k + 1];
                        reinterpret_cast<typename Vec4<T>::type*>(row)[k / 2] = v4;
                    }
                    if (dim == 0) {
                        int cx, cy, cz;
                        unpack_cell(sl.cell, cx, cy, cz);
                        int zrel = cz - tz0;              // trimmed bins: c_z may be the first plane of the next tile
                        zrel += zrel < 0 ? g.n : 0;
                        cx += pr.dx > (T)0 ? 1 : 0; cy += pr.dy > (T)0 ? 1 : 0; zrel += pr.dz > (T)0 ? 1 : 0;
                        base_s[slot] = zrel * SPL + (cy - ty0) * SX + (cx - tx0) + (C::XS - M_);
                        q_s[slot] = pre * pr.q;
                        idx_s[slot] = (int)sl.idx;
                    }
                }
                if (!tile_ready) {                   // the first batch's weights overlapped the tile copy
                    cp_async_wait_all();
                    __syncthreads();
                    tile_ready = true;
                } else {
                    __syncwarp();
                }
                // ---- pairs: half-warp h contracts particle pr + h
                for (int pr2 = 0; pr2 < nb; pr2 += 2) {
                    const bool act = pr2 + half < nb;
                    const int slot = act ? pr2 + half : pr2;     // an idle half repeats its neighbour's particle, result dropped
                    const P2* wt = wtab + slot * 3 * WP;
                    P2 wx[WE], wy[NR], wz[NR];
                    {
                        using V4 = typename Vec4<T>::type;
                        const V4* w4 = reinterpret_cast<const V4*>(wt);
#pragma unroll
                        for (int v = 0; v < WE / 2; ++v) {
                            const V4 t4 = w4[v];
                            wx[2 * v].x = t4.x; wx[2 * v].y = t4.y; wx[2 * v + 1].x = t4.z; wx[2 * v + 1].y = t4.w;
                        }
                    }
#pragma unroll
                    for (int i = 0; i < NR; ++i) { wy[i] = wt[WP + ya + 4 * i]; wz[i] = wt[2 * WP + zb + 4 * i]; }
                    const int base = base_s[slot];
                    const T* origin = tile_s + base + rowbase;
                    T fx = (T)0, fy = (T)0, fz = (T)0;
                    // (sum Psi phi_x, sum Psi phi_x') of one row -> the three force sums with the row's y, z weights
                    auto finish_sums = [&](int i, int j, const P2 s2) {
                        if (kIk) {
                            fx += s2.x * (wy[i].x * wz[j].x);
                        } else {
                            const P2 yz = pair_scale(wy[i], wz[j].x);      // (phi_y phi_z, phi_y' phi_z)
                            fx += s2.y * yz.x;
                            fy += s2.x * yz.y;
                            fz += s2.x * (wy[i].x * wz[j].y);
                        }
                    };
                    if ((base & 1) == 0) {
#pragma unroll
                        for (int j = 0; j < NR; ++j)
#pragma unroll
                            for (int i = 0; i < NR; ++i) {
                                const P2* row = reinterpret_cast<const P2*>(origin + 4 * i * SX + 4 * j * SPL);
                                P2 sa, sb2; sa.x = (T)0; sa.y = (T)0; sb2.x = (T)0; sb2.y = (T)0;
#pragma unroll
                                for (int k = 0; k < WE / 2; ++k) {
                                    const P2 t2 = row[k];
                                    fma_pair(sa, wx[2 * k], t2.x);
                                    fma_pair(sb2, wx[2 * k + 1], t2.y);
                                }
                                finish_sums(i, j, pair_add(sa, sb2));
                            }
                    } else {
                        // the row starts on an odd column: first and last element by single-word loads, the rest as
                        // aligned pairs.  A single-word load serves both halves in one wavefront only if they hit
                        // different banks: the 16 first elements of a half sit in the 16 odd banks, the 16 last ones
                        // in the 16 even banks, so half 0 loads (first, last) and half 1 (last, first)
                        const P2 wa = half ? wx[WE - 1] : wx[0], wb = half ? wx[0] : wx[WE - 1];
                        const int oa = half ? WE - 1 : 0, ob = half ? 0 : WE - 1;
#pragma unroll
                        for (int j = 0; j < NR; ++j)
#pragma unroll
                            for (int i = 0; i < NR; ++i) {
                                const T* rowf = origin + 4 * i * SX + 4 * j * SPL;
                                const P2* row = reinterpret_cast<const P2*>(rowf + 1);
                                P2 sa, sb2; sa.x = (T)0; sa.y = (T)0; sb2.x = (T)0; sb2.y = (T)0;
                                fma_pair(sa, wa, rowf[oa]);
#pragma unroll
                                for (int k = 0; k < WE / 2 - 1; ++k) {
                                    const P2 t2 = row[k];
                                    fma_pair(sb2, wx[2 * k + 1], t2.x);
                                    fma_pair(sa, wx[2 * k + 2], t2.y);
                                }
                                fma_pair(sb2, wb, rowf[ob]);
                                finish_sums(i, j, pair_add(sa, sb2));
                            }
                    }
                    const size_t jp = (size_t)(uint32_t)idx_s[slot];
                    const T sc = q_s[slot];
                    if (kIk) {
#pragma unroll
                        for (int o = 8; o > 0; o >>= 1) fx += __shfl_xor_sync(0xffffffffu, fx, o);
                        if (act && l16 == 0) F[3 * jp + component] = sc * fx;
                    } else {
                        // the three sums over the 16 lanes of the half by recursive halving (5 shuffles); the totals of
                        // x, y, z end in the lanes l16 = 0, 4, 8
                        const bool b3 = (l16 & 8) != 0, b2 = (l16 & 4) != 0;
                        const T k0 = (b3 ? fz : fx) + __shfl_xor_sync(0xffffffffu, b3 ? fx : fz, 8);
                        const T k1 = (b3 ? (T)0 : fy) + __shfl_xor_sync(0xffffffffu, b3 ? fy : (T)0, 8);
                        T kk = (b2 ? k1 : k0) + __shfl_xor_sync(0xffffffffu, b2 ? k0 : k1, 4);
                        kk += __shfl_xor_sync(0xffffffffu, kk, 2);
                        kk += __shfl_xor_sync(0xffffffffu, kk, 1);
                        // (ry, rz: the y and z prefactors of an orthorhombic box relative to x; 1 otherwise)
                        if (act && (l16 & 3) == 0 && l16 < 12) F[3 * jp + (l16 >> 2)] = sc * kk * (l16 < 4 ? (T)1 : (l16 < 8 ? ry : rz));
                    }
                }
                __syncwarp();                        // the batch's weight rows are rewritten next
            }
        }
        if (!tile_ready) { cp_async_wait_all(); __syncthreads(); }   // (a warp without particles still joins the barrier)
        return;
    }

    // stencil rows owned by this lane: rr = lane + 32 it -> (rz, ry)
    int rowoff[ITER], ryo[ITER], rzo[ITER];
#pragma unroll
    for (int it = 0; it < ITER; ++it) {
        const int rr = lane + 32 * it;
        const int rz = rr / WE, ry = rr - rz * WE;
        rowoff[it] = rz * SPL + ry * SX;
        ryo[it] = WP + ry;          // index into the particle's [3][WP] weight rows
        rzo[it] = 2 * WP + rz;
    }

    P2* wtab = wtab_all + warp * PBW * 3 * WP;
    T* q_s = q_all + warp * PBW;
    int* base_s = base_all + warp * PBW;
    int* idx_s = idx_all + warp * PBW;
    // window values of one warp batch: one lane per (dimension, particle)
    auto batch_weights = [&](int p0, int nb) {
        if (lane < 3 * nb) {
            const int dim = lane / nb, slot = lane - dim * nb;
            const uint32_t gi = slot_of(p0 + slot);
            const PRec<T> pr = slots[gi].rec;
            const T d0 = dim == 0 ? pr.dx : (dim == 1 ? pr.dy : pr.dz);
            T w[W], dw[W];
            stencil_weights<T, M_, !kIk, true>(wp, pa, d0, w, dw);   // packed Horner chains
            P2* row = wtab + (slot * 3 + dim) * WP;
            const bool sh = kTrim && d0 > (T)0;                 // ks = 1: the k = 0 point is the zero one
#pragma unroll
            for (int k = 0; k < WE; ++k) {
                P2 v;
                v.x = (kTrim && sh) ? w[k + (kTrim ? 1 : 0)] : w[k];
                v.y = (kTrim && sh) ? dw[k + (kTrim ? 1 : 0)] : dw[k];
                row[k] = v;
            }
            if (dim == 0) {
                int cx, cy, cz;
                unpack_cell(slots[gi].cell, cx, cy, cz);
                int zrel = cz - tz0;                  // trimmed bins: c_z may be the first plane of the next tile
                zrel += zrel < 0 ? g.n : 0;
                if (kTrim) {
                    cx += pr.dx > (T)0 ? 1 : 0; cy += pr.dy > (T)0 ? 1 : 0; zrel += pr.dz > (T)0 ? 1 : 0;
                }
                base_s[slot] = zrel * SPL + (cy - ty0) * SX + (cx - tx0) + (C::XS - M_);
                q_s[slot] = pre * pr.q;
                idx_s[slot] = (int)slots[gi].idx;
            }
        }
    };

    // the first batch's weights overlap the tile copy
    // every warp takes one contiguous share of the tile's particles (sizes differ by at most one), in
    // batches of PBW: the CTA ends within one particle of perfect balance
    const int share = cnt / C::WARPS, extra = cnt - share * C::WARPS;
    const int wbeg = warp * share + min(warp, extra), wend = wbeg + share + (warp < extra ? 1 : 0);
    if (wbeg < wend) batch_weights(wbeg, min(PBW, wend - wbeg));
    cp_async_wait_all();
    __syncthreads();

    for (int p0 = wbeg; p0 < wend; p0 += PBW) {
        const int nb = min(PBW, wend - p0);
        if (p0 != wbeg) {
            batch_weights(p0, nb);
            __syncwarp();
        }
        // ---- one particle after the other
        for (int slot = 0; slot < nb; ++slot) {
            const P2* wt = wtab + slot * 3 * WP;
            P2 wx[WE + 1];
            {
                using V4 = typename Vec4<T>::type;
                const V4* w4 = reinterpret_cast<const V4*>(wt);
#pragma unroll
                for (int v = 0; v < (WE + 1) / 2; ++v) {
                    const V4 t4 = w4[v];
                    wx[2 * v].x = t4.x; wx[2 * v].y = t4.y; wx[2 * v + 1].x = t4.z; wx[2 * v + 1].y = t4.w;
                }
            }
            const int base = base_s[slot];
            const T* origin = tile_s + base;
            // kWide (fp32, analytic variant, m <= 3): the three sums are formed in fp64.  sum Psi phi' cancels
            // heavily and the narrow windows have twice the max|phi'| of m >= 4, so the fp32 summation error
            // alone reaches the 2e-6 bar there; the stencil is small, the fp64 FMAs are cheap.
            constexpr bool kWide = sizeof(T) == 4 && M_ <= 3 && !kIk;
            using A = typename std::conditional<kWide, double, T>::type;
            A fx = (A)0, fy = (A)0, fz = (A)0;
            // one stencil row: s = sum_k (phi, phi')[k] * v[k], then the y, z weights of the row
            auto finish_row = [&](int it, const T (&v)[WE]) {
                const P2 wy = wt[ryo[it]], wz = wt[rzo[it]];
                if constexpr (kWide) {
                    double s0 = 0.0, s1 = 0.0;
#pragma unroll
                    for (int k = 0; k < WE; ++k) {
                        s0 = fma((double)wx[k].x, (double)v[k], s0);
                        s1 = fma((double)wx[k].y, (double)v[k], s1);
                    }
                    fx = fma(s1, (double)wy.x * (double)wz.x, fx);
                    fy = fma(s0, (double)wy.y * (double)wz.x, fy);
                    fz = fma(s0, (double)wy.x * (double)wz.y, fz);
                } else {
                    P2 sa, sb2; sa.x = (T)0; sa.y = (T)0; sb2.x = (T)0; sb2.y = (T)0;
#pragma unroll
                    for (int k = 0; k < WE; ++k) {
                        if (k & 1) fma_pair(sb2, wx[k], v[k]);
                        else fma_pair(sa, wx[k], v[k]);
                    }
                    const P2 s2 = pair_add(sa, sb2);                   // (sum Psi phi_x, sum Psi phi_x')
                    if (kIk) {
                        fx += s2.x * (wy.x * wz.x);
                    } else {
                        const P2 yz = pair_scale(wy, wz.x);            // (phi_y phi_z, phi_y' phi_z)
                        fx += s2.y * yz.x;
                        fy += s2.x * yz.y;
                        fz += s2.x * (wy.x * wz.y);
                    }
                }
            };
            if constexpr (C::kPair && sizeof(T) == 4) {
                // 8-byte loads of aligned pairs; the row starts on an even or an odd column (warp-uniform)
                if ((base & 1) == 0) {
#pragma unroll
                    for (int it = 0; it < ITER; ++it) {
                        if (it + 1 < ITER || lane + 32 * it < WE * WE) {
                            const P2* row = reinterpret_cast<const P2*>(origin + rowoff[it]);
                            T v[WE];
#pragma unroll
                            for (int j = 0; j < WE / 2; ++j) { const P2 t2 = row[j]; v[2 * j] = t2.x; v[2 * j + 1] = t2.y; }
                            finish_row(it, v);
                        }
                    }
                } else {
#pragma unroll
                    for (int it = 0; it < ITER; ++it) {
                        if (it + 1 < ITER || lane + 32 * it < WE * WE) {
                            const T* rowf = origin + rowoff[it];
                            const P2* row = reinterpret_cast<const P2*>(rowf + 1);
                            T v[WE];
                            v[0] = rowf[0];
#pragma unroll
                            for (int j = 0; j < WE / 2 - 1; ++j) { const P2 t2 = row[j]; v[2 * j + 1] = t2.x; v[2 * j + 2] = t2.y; }
                            v[WE - 1] = rowf[WE - 1];
                            finish_row(it, v);
                        }
                    }
                }
            } else {
#pragma unroll
                for (int it = 0; it < ITER; ++it) {
                    if (it + 1 < ITER || lane + 32 * it < WE * WE) {
                        const T* row = origin + rowoff[it];
                        T v[WE];
#pragma unroll
                        for (int k = 0; k < WE; ++k) v[k] = row[k];
                        finish_row(it, v);
                    }
                }
            }
            const size_t j = (size_t)(uint32_t)idx_s[slot];
            const T sc = q_s[slot];
            if (kIk) {
#pragma unroll
                for (int o = 16; o > 0; o >>= 1) fx += __shfl_xor_sync(0xffffffffu, fx, o);
                if (lane == 0) F[3 * j + component] = sc * fx;
            } else {
                // the three sums by recursive halving: (fx, fy | fz, -) over lane bit 4, then one value per
                // lane over bit 3, then a plain butterfly: 6 shuffles instead of 15.  The totals of x, y, z
                // end in the lanes with (lane >> 3) = 0, 1, 2.
                const bool b4 = (lane & 16) != 0, b3 = (lane & 8) != 0;
                A k0 = (b4 ? fz : fx) + __shfl_xor_sync(0xffffffffu, b4 ? fx : fz, 16);
                A k1 = (b4 ? (A)0 : fy) + __shfl_xor_sync(0xffffffffu, b4 ? fy : (A)0, 16);
                A k = (b3 ? k1 : k0) + __shfl_xor_sync(0xffffffffu, b3 ? k0 : k1, 8);
                k += __shfl_xor_sync(0xffffffffu, k, 4);
                k += __shfl_xor_sync(0xffffffffu, k, 2);
                k += __shfl_xor_sync(0xffffffffu, k, 1);
                if ((lane & 7) == 0 && lane < 24) F[3 * j + (lane >> 3)] = (T)((A)sc * k) * (lane < 8 ? (T)1 : (lane < 16 ? ry : rz));
            }
        }
        __syncwarp();
    }
}

}  // namespace enuf
