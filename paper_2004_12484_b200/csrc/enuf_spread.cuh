// Step a2 -- spreading (adjoint NFFT, part 1):
//   g[l] = sum_j q_j phi(u_jx - l_x) phi(u_jy - l_y) phi(u_jz - l_z), l periodic.
//
// Output-stationary, sliding z-window, warp-specialised.  A CTA owns a column of CX x 16 grid cells in
// (x, y) (CX = 32, or 16 on small grids) and a chunk [z0, z1) of grid planes.  It has
//   - NCONS = CX/8 x 2 CONSUMER warps, each owning an 8 x 8 patch of the column: every lane owns two
//     x-adjacent cells and keeps, in registers, their partial sums on the WZ consecutive planes that the
//     particles of slab s (bin plane s) can reach.  Per (warp, particle) visit the work is WZ packed FMAs
//     acc[k] += (a0, a1) * (q wz[k]) with (a0, a1) = wx[cells] * wy[cell].  After slab s the lowest plane
//     of the window is complete: one coalesced store, and the window slides.  Every grid value is written
//     exactly once -- no atomics, no clearing of the grid, no shared-memory read-modify-write;
//   - two PRODUCER warps, one per stage of a two-stage buffer in shared memory, taking the slabs in turn:
//     a producer culls the particles of the neighbouring bins against the column's halo, copies the three
//     window rows of the accepted ones (3 x 16 values, evaluated ONCE per particle by the bin scatter --
//     "window values computed [once and kept]") into slots of its stage with cp.async, builds
//     for every patch the list of staged particles whose stencil overlaps it, and hands the stage over
//     through an mbarrier (full / empty pair per stage; the copies arrive on the full barrier themselves).
//     The consumers never meet at a CTA-wide barrier: each waits only for the producers, and hands a
//     stage back when its own visits are done.
//
// Stage layout.  One slot per staged particle, PITCH = 68 elements (76 for 13-point stencils):
//   [0,8) zeros | [8,24) x row | zeros | [OYF, OYF+16) y row | zeros | [OZF, OZF+16) q * z row
// The rows are placed RELATIVE TO THE STENCIL, not to the column: a lane of the patch with origin (px0, py0)
// whose cells are lxl, lxl + 1 (lxl even) and row lyl reads
//   wx pair at 8 + par + px0 - X0 + lxl,   wy at OYF + py0 - Y0 + lyl      (X0, Y0: first stencil point, column coords)
// -- for a patch the stencil overlaps, px0 - X0 lies in [-7, WZ - 1], so the index stays inside the slot's
// zero padding, and lanes outside the stencil read zeros.  par = X0 & 1 shifts the x row by one element so
// that the pair is always 8-byte aligned.  The visit lists carry these addresses ready-made.
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

// kTrim (fp32 Kaiser-Bessel, m >= 5): particles are binned by the plane s = c_z - 1 + ks_z, ks = (d0 > 0),
// so that every particle of slab s has its 2m non-zero z weights on the planes s-m+1 .. s+m: the window
// is WZ = 2m planes and the x / y stencils are the 2m points from c - m + ks on.
template <typename T, int M_, bool kTrim, int NPX_>
struct SpreadCfg {
    static constexpr int W = 2 * M_ + 1;
    static constexpr int WZ = W - (kTrim ? 1 : 0);               // stencil points per dimension = planes in the window
    static constexpr int SLO = M_, SHI = kTrim ? M_ - 1 : M_;    // slab s reaches the planes s - SHI .. s + SLO
    static constexpr int NPX = NPX_, NPY = 2, NCONS = NPX * NPY; // 8 x 8 patches = consumer warps
    static constexpr int NPROD = 2;                              // producer warps = stages: producer k fills stage k
    static constexpr int CX = 8 * NPX, CY = 8 * NPY;             // column
    static constexpr int NT = 32 * (NCONS + NPROD);
    static constexpr int NBX = CX / kTile + 2, NBY = CY / kTile + 2;   // bins (16 x 16, enuf_common.cuh) the halo touches
    static constexpr int NBIN = NBX * NBY, NPAIR = (NBIN + 1) / 2;
    // slot layout (elements of T): zeros | x row | zeros | y row | zeros | z row ; the largest index a lane reads is
    // x: 8 + 1 + (WZ-1) + 7, y: OYF + (WZ-1) + 7 (header comment)
    static constexpr int OXF = 8;
    static constexpr int OYF = (16 + WZ + 3) / 4 * 4 > 24 ? (16 + WZ + 3) / 4 * 4 : 24;
    static constexpr int OZF = (OYF + WZ + 7 + 3) / 4 * 4 > OYF + 16 ? (OYF + WZ + 7 + 3) / 4 * 4 : OYF + 16;
    static constexpr int PITCH = OZF + 16 <= 68 ? 68 : 76;       // = 4 / 12 mod 32: 16-byte row chunks of 8 slots hit 32 banks
    static constexpr int CAP = sizeof(T) == 4 ? (NPX == 4 ? (PITCH == 68 ? 96 : 88) : 56) : (NPX == 4 ? 48 : 40);   // staged particles per round
    static constexpr int LCAP = CAP + 4;                         // visit-list entries per patch (even padding + prefetch)
    static constexpr int NSTAGE = NPROD;
    static constexpr int kBlk = 16;                              // slabs (of one producer) whose bin ranges are loaded at once
    static constexpr int CTAS_PER_SM = sizeof(T) == 4 ? (NPX == 4 ? 3 : 5) : (NPX == 4 ? 1 : 2);
    static constexpr size_t SLOT_BYTES = sizeof(T) * (size_t)(CAP + 1) * PITCH;   // slot CAP is all zero
    static constexpr size_t LIST_BYTES = sizeof(uint2) * (size_t)NCONS * LCAP;
    static constexpr size_t STAGE_BYTES = ((SLOT_BYTES + LIST_BYTES + sizeof(int) * CAP + 15) / 16) * 16;
    static_assert(CAP >= 32, "a cull step stages up to 32 particles");
    static_assert(SLOT_BYTES < 65536, "visit-list entries are 16-bit byte offsets");
    static_assert(OZF + 16 <= PITCH, "slot layout");
};

template <typename T, int M_, bool kTrim, int NPX>
constexpr size_t spread_smem_bytes() {
    using C = SpreadCfg<T, M_, kTrim, NPX>;
    return C::STAGE_BYTES * C::NSTAGE;
}

// The three 16-element window rows of one particle, as the spreading kernel stages them (written once per
// particle by the bin scatter, enuf_bin.cuh, read by every CTA whose halo the particle is in):
//   x row: element j = phi_x at stencil point j - parx (parx = parity of the first stencil point's grid index),
//   y row: element j = phi_y at stencil point j,   z row: element j = q phi_z at stencil point j,
// zero beyond the WZ stencil points.  kTrim: stencil point k is point k + ks of the 2m+1 (ks = d0 > 0).
constexpr int kRowElems = 16, kRowsPerParticle = 3;
template <typename T, int M_, bool kTrim>
__device__ __forceinline__ void write_window_rows(const WindowParams& wp, const PolyArg<M_>& pa, T dx, T dy, T dz, T q,
                                                  int parx, T* __restrict__ dst) {
    constexpr int W = 2 * M_ + 1, WZ = W - (kTrim ? 1 : 0);
    using V4 = typename Vec4<T>::type;
#pragma unroll
    for (int dim = 0; dim < 3; ++dim) {
        const T d0 = dim == 0 ? dx : (dim == 1 ? dy : dz);
        T w[W], dw[W];
        stencil_weights<T, M_, false>(wp, pa, d0, w, dw);
        const int sh = (kTrim && d0 > (T)0) ? 1 : 0;
        const int par = dim == 0 ? parx : 0;
        const T mult = dim == 2 ? q : (T)1;
        T r16[kRowElems];
#pragma unroll
        for (int j = 0; j < kRowElems; ++j) {
            // element j holds stencil point k = j - par, i.e. w[k + sh]
            T v = (T)0;
            if (kTrim) {
                const T a0 = (j < WZ) ? w[j < W ? j : 0] : (T)0;                          // par 0, sh 0
                const T a1 = (j + 1 < W && j < WZ) ? w[j + 1 < W ? j + 1 : 0] : (T)0;      // par 0, sh 1
                const T b0 = (j >= 1 && j - 1 < WZ) ? w[j >= 1 ? j - 1 : 0] : (T)0;        // par 1, sh 0
                const T b1 = (j >= 1 && j - 1 < WZ) ? w[j < W ? j : 0] : (T)0;             // par 1, sh 1
                v = par ? (sh ? b1 : b0) : (sh ? a1 : a0);
            } else {
                const T a0 = (j < WZ) ? w[j < W ? j : 0] : (T)0;
                const T b0 = (j >= 1 && j - 1 < WZ) ? w[j >= 1 ? j - 1 : 0] : (T)0;
                v = par ? b0 : a0;
            }
            r16[j] = v * mult;
        }
        V4* row4 = reinterpret_cast<V4*>(dst + dim * kRowElems);
#pragma unroll
        for (int v = 0; v < kRowElems / 4; ++v) {
            V4 o; o.x = r16[4 * v]; o.y = r16[4 * v + 1]; o.z = r16[4 * v + 2]; o.w = r16[4 * v + 3];
            row4[v] = o;
        }
    }
}

__device__ __forceinline__ void cp_async_16(uint32_t smem_dst, const void* gmem_src) {
    asm volatile("cp.async.cg.shared.global [%0], [%1], 16;" ::"r"(smem_dst), "l"(gmem_src) : "memory");
}
// the mbarrier receives one arrival when all cp.async operations this thread has issued so far are complete
__device__ __forceinline__ void cp_async_mbar_arrive(uint64_t* bar) {
    asm volatile("cp.async.mbarrier.arrive.noinc.shared::cta.b64 [%0];" ::"r"(smem_u32(bar)) : "memory");
}

// slots[].cell: bits 0..29 the packed nearest cell, bits 30 / 31 = ks_x / ks_y (trimmed plans; enuf_bin.cuh)
// rows: [N][3][16] window rows in bin order (write_window_rows)
template <typename T, int M_, bool kTrim, int NPX>
__global__ void __launch_bounds__((SpreadCfg<T, M_, kTrim, NPX>::NT), (SpreadCfg<T, M_, kTrim, NPX>::CTAS_PER_SM))
spread_kernel(const PSlot<T>* __restrict__ slots, const T* __restrict__ rows,
              const uint32_t* __restrict__ offset, TileGeom g, int zchunk, T* __restrict__ grid) {
    using C = SpreadCfg<T, M_, kTrim, NPX>;
    using P2 = typename Pair2<T>::type;
    using V4 = typename Vec4<T>::type;
    constexpr int WZ = C::WZ, NCONS = C::NCONS, CX = C::CX, CY = C::CY, CAP = C::CAP, LCAP = C::LCAP;
    constexpr int PITCH = C::PITCH, OXF = C::OXF, OYF = C::OYF, OZF = C::OZF;
    constexpr int NBX = C::NBX, NBIN = C::NBIN, NPAIR = C::NPAIR, NSTAGE = C::NSTAGE, kBlk = C::kBlk;
    constexpr unsigned ES = (unsigned)sizeof(T);
    constexpr unsigned FULL = 0xffffffffu;
    constexpr int NCH = (int)(kRowElems * sizeof(T) / 16);        // 16-byte chunks per row

    extern __shared__ __align__(16) unsigned char smem_raw[];
    __shared__ uint64_t full_bar[NSTAGE], empty_bar[NSTAGE];
    __shared__ int cnt_s[NSTAGE][NCONS];        // visits of each patch in the stage (even, zero-record padded)
    __shared__ int last_s[NSTAGE];              // 1: the stage is the last round of its slab
    __shared__ uint32_t rng[C::NPROD][NBIN][2 * kBlk];   // [..][0..kBlk): range starts of kBlk slabs, [kBlk..): ends

    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    constexpr int ncx_per = CX / kTile, ncy_per = CY / kTile;
    const int ncolx = g.n / CX;
    const int Tx = blockIdx.x % ncolx, Ty = blockIdx.x / ncolx;
    const int z0 = blockIdx.y * zchunk, z1 = min(g.n, z0 + zchunk);
    const int s_begin = z0 - C::SLO, s_end = z1 + C::SHI;

    // the zero padding of every slot (and the all-zero slot CAP) is written once; rows are rewritten per round
    for (int i = tid; i < (int)(C::STAGE_BYTES * NSTAGE / 16); i += C::NT)
        reinterpret_cast<uint4*>(smem_raw)[i] = make_uint4(0u, 0u, 0u, 0u);
    if (tid == 0) {
#pragma unroll
        for (int st = 0; st < NSTAGE; ++st) {
            // full: one arrival per producer lane when its row copies have landed + one after the lists are written
            mbar_init(&full_bar[st], 33);
            mbar_init(&empty_bar[st], NCONS);
        }
    }
    __syncthreads();

    if (warp >= NCONS) {
        // =========================================================== producers
        // producer k fills stage k with the slabs s_begin + k, s_begin + k + 2, ..
        const int k = warp - NCONS, stage = k;
        const int half = lane >> 4, l16 = lane & 15;
        const unsigned below = (1u << lane) - 1u;
        int bin0 = 0;                            // lane b < NBIN: first bin (plane 0) of neighbouring bin column b
        if (lane < NBIN) {
            int tbx = Tx * ncx_per - 1 + lane % NBX, tby = Ty * ncy_per - 1 + lane / NBX;
            tbx += tbx < 0 ? g.nt : 0; tbx -= tbx >= g.nt ? g.nt : 0;
            tby += tby < 0 ? g.nt : 0; tby -= tby >= g.nt ? g.nt : 0;
            bin0 = (tby * g.nt + tbx) * g.n;
        }
        unsigned char* sbase = smem_raw + (size_t)stage * C::STAGE_BYTES;
        const uint32_t sl32 = smem_u32(sbase);
        uint2* lists = reinterpret_cast<uint2*>(sbase + C::SLOT_BYTES);
        int* pk = reinterpret_cast<int*>(sbase + C::SLOT_BYTES + C::LIST_BYTES);
        uint32_t (*rg)[2 * kBlk] = rng[k];
        unsigned pe = 0;                         // phase of empty_bar[stage] this producer waits for next, flipped
        int blk0 = s_begin + k - 2 * kBlk;
        for (int s = s_begin + k; s < s_end; s += C::NPROD) {
            if (s - blk0 >= 2 * kBlk) {
                // ranges of this producer's next kBlk slabs: lane & 15 = slab, lanes 0..15 load the starts, 16..31 the ends
                blk0 = s;
                __syncwarp();
                const int cz = (blk0 + 2 * l16) & (g.n - 1);
#pragma unroll
                for (int b = 0; b < NBIN; ++b) {
                    const int bb = __shfl_sync(FULL, bin0, b);
                    rg[b][lane] = offset[bb + cz + half];
                }
                __syncwarp();
            }
            const int js = (s - blk0) >> 1;
            int c0 = 0, p0 = 0;                  // next candidates: index c0 + (0..15) of the bins of pairs p0..
            bool slab_done = false;
            while (!slab_done) {
                mbar_wait(&empty_bar[stage], pe ^ 1u);
                pe ^= 1u;
                int ns = 0;
                // ---- cull: 16 candidates of two bins per step (half-warp each); all cell loads of a sweep over
                //      the bins are issued before the first is examined.  An accepted particle's three window
                //      rows are copied from global memory into its slot by cp.async.
                for (;;) {
                    uint32_t cellw[NPAIR], pidx[NPAIR];
                    int cmax = 0;
#pragma unroll
                    for (int p = 0; p < NPAIR; ++p) {
                        const int b = 2 * p + half;
                        uint32_t st = 0; int cn = 0;
                        if (b < NBIN) { st = rg[b][js]; cn = (int)(rg[b][kBlk + js] - st); }
                        cmax = max(cmax, cn);
                        const int kk = c0 + l16;
                        pidx[p] = st + (uint32_t)kk;
                        cellw[p] = (p >= p0 && kk < cn) ? slots[pidx[p]].cell : 0xffffffffu;
                    }
                    cmax = max(cmax, __shfl_xor_sync(FULL, cmax, 16));
                    bool stop = false;
#pragma unroll
                    for (int p = 0; p < NPAIR; ++p) {
                        if (p < p0) continue;
                        const uint32_t cw = cellw[p];
                        const unsigned vb = __ballot_sync(FULL, cw != 0xffffffffu);
                        if (vb == 0u) continue;                       // both bins exhausted
                        if (ns + __popc(vb) > CAP) { p0 = p; stop = true; break; }
                        const int b = 2 * p + half;
                        // first stencil point, column coords: nearest cell - m (+ ks when trimmed)
                        const int X0 = (int)(cw & 15u) + (b % NBX - 1) * kTile - M_ + (kTrim ? (int)((cw >> 30) & 1u) : 0);
                        const int Y0 = (int)((cw >> 10) & 15u) + (b / NBX - 1) * kTile - M_ + (kTrim ? (int)(cw >> 31) : 0);
                        const bool ok = cw != 0xffffffffu && X0 <= CX - 1 && X0 + WZ - 1 >= 0 && Y0 <= CY - 1 && Y0 + WZ - 1 >= 0;
                        const unsigned bal = __ballot_sync(FULL, ok);
                        if (ok) {
                            const int pos = ns + __popc(bal & below);
                            pk[pos] = (X0 + 32) | ((Y0 + 32) << 8);
                            const char* src = reinterpret_cast<const char*>(rows + (size_t)pidx[p] * (kRowsPerParticle * kRowElems));
                            const uint32_t dst = sl32 + (uint32_t)(pos * PITCH) * ES;
#pragma unroll
                            for (int c = 0; c < NCH; ++c) cp_async_16(dst + OXF * ES + 16 * c, src + 16 * c);
#pragma unroll
                            for (int c = 0; c < NCH; ++c) cp_async_16(dst + OYF * ES + 16 * c, src + 16 * (NCH + c));
#pragma unroll
                            for (int c = 0; c < NCH; ++c) cp_async_16(dst + OZF * ES + 16 * c, src + 16 * (2 * NCH + c));
                        }
                        ns += __popc(bal);
                    }
                    if (stop) break;
                    p0 = 0; c0 += 16;
                    if (c0 >= cmax) { slab_done = true; break; }
                }
                cp_async_mbar_arrive(&full_bar[stage]);
                __syncwarp();
                // ---- visit lists: for every patch the staged particles whose stencil overlaps it, as ready-made
                //      byte offsets (x row | z row << 16, y row) into the stage
                int lc[NCONS];
#pragma unroll
                for (int w8 = 0; w8 < NCONS; ++w8) lc[w8] = 0;
                for (int g0 = 0; g0 < ns; g0 += 32) {
                    const int slot = g0 + lane;
                    const bool v = slot < ns;
                    int X0 = 64, Y0 = 64;
                    if (v) { const int pkv = pk[slot]; X0 = (pkv & 255) - 32; Y0 = ((pkv >> 8) & 255) - 32; }
                    const unsigned sb = (unsigned)(slot * PITCH) * ES;
                    const unsigned xb = sb + (unsigned)(OXF + (X0 & 1) - X0) * ES;
                    const unsigned yb = sb + (unsigned)(OYF - Y0) * ES;
                    const unsigned zb = sb + (unsigned)OZF * ES;
#pragma unroll
                    for (int w8 = 0; w8 < NCONS; ++w8) {
                        const int px0 = 8 * (w8 % NPX), py0 = 8 * (w8 / NPX);
                        const bool ov = v && X0 <= px0 + 7 && X0 + WZ - 1 >= px0 && Y0 <= py0 + 7 && Y0 + WZ - 1 >= py0;
                        const unsigned bal = __ballot_sync(FULL, ov);
                        if (ov) lists[w8 * LCAP + lc[w8] + __popc(bal & below)] =
                                    make_uint2((xb + (unsigned)px0 * ES) | (zb << 16), yb + (unsigned)py0 * ES);
                        lc[w8] += __popc(bal);
                    }
                }
                if (lane == 0) {
                    const unsigned zs = (unsigned)(CAP * PITCH) * ES;      // the all-zero slot
#pragma unroll
                    for (int w8 = 0; w8 < NCONS; ++w8) {
                        int c = lc[w8];
                        if (c & 1) { lists[w8 * LCAP + c] = make_uint2((zs + OXF * ES) | ((zs + OZF * ES) << 16), zs + OYF * ES); ++c; }
                        cnt_s[stage][w8] = c;
                    }
                    last_s[stage] = slab_done ? 1 : 0;
                }
                __threadfence_block();
                __syncwarp();
                if (lane == 0) mbar_arrive(&full_bar[stage]);
            }
        }
        return;
    }

    // =============================================================== consumers
    const int px0 = 8 * (warp % NPX), py0 = 8 * (warp / NPX);
    const int lxl = (lane & 3) * 2, lyl = lane >> 2;              // this lane's two cells (lxl, lyl), (lxl + 1, lyl) of the patch
    T* gout = grid + ((size_t)(Ty * CY + py0 + lyl)) * g.n + Tx * CX + px0 + lxl;
    const size_t plane = (size_t)g.n * g.n;

    P2 acc[WZ];
#pragma unroll
    for (int k = 0; k < WZ; ++k) { acc[k].x = (T)0; acc[k].y = (T)0; }

    unsigned pf = 0;                                              // phase bits of full_bar[0], full_bar[1]
    for (int s = s_begin; s < s_end; ++s) {
        const int stage = (s - s_begin) & 1;
        const unsigned char* sbase = smem_raw + (size_t)stage * C::STAGE_BYTES;
        const char* sbx = reinterpret_cast<const char*>(sbase) + lxl * ES;
        const char* sby = reinterpret_cast<const char*>(sbase) + lyl * ES;
        const char* sbz = reinterpret_cast<const char*>(sbase);
        const uint4* lp = reinterpret_cast<const uint4*>(sbase + C::SLOT_BYTES) + warp * (LCAP / 2);
        int lastf;
        do {
            mbar_wait(&full_bar[stage], (pf >> stage) & 1u);
            pf ^= 1u << stage;
            const int cnt = cnt_s[stage][warp];
            lastf = last_s[stage];
            uint4 ee = lp[0];
            for (int i = 0; i < cnt; i += 2) {
                const uint4 e = ee;
                ee = lp[(i >> 1) + 1];                                   // next trip (the list has spare entries)
                const P2 wx1 = *reinterpret_cast<const P2*>(sbx + (e.x & 0xffffu));
                const T wy1 = *reinterpret_cast<const T*>(sby + e.y);
                const P2 wx2 = *reinterpret_cast<const P2*>(sbx + (e.z & 0xffffu));
                const T wy2 = *reinterpret_cast<const T*>(sby + e.w);
                constexpr int NV = (WZ + 3) / 4;
                V4 zv1[NV], zv2[NV];
#pragma unroll
                for (int v = 0; v < NV; ++v) zv1[v] = reinterpret_cast<const V4*>(sbz + (e.x >> 16))[v];
#pragma unroll
                for (int v = 0; v < NV; ++v) zv2[v] = reinterpret_cast<const V4*>(sbz + (e.z >> 16))[v];
                const P2 a1 = pair_scale(wx1, wy1), a2 = pair_scale(wx2, wy2);
                const T* wz1 = reinterpret_cast<const T*>(zv1);
                const T* wz2 = reinterpret_cast<const T*>(zv2);
#pragma unroll
                for (int k = 0; k < WZ; ++k) fma_pair(acc[k], a1, wz1[k]);
#pragma unroll
                for (int k = 0; k < WZ; ++k) fma_pair(acc[k], a2, wz2[k]);
            }
            __syncwarp();
            if (lane == 0) mbar_arrive(&empty_bar[stage]);
        } while (!lastf);
        // the lowest plane of the window (s - SHI) is complete: store it, slide
        const int zo = s - C::SHI;
        if (zo >= z0) *reinterpret_cast<P2*>(gout + (size_t)zo * plane) = acc[0];
#pragma unroll
        for (int k = 0; k + 1 < WZ; ++k) acc[k] = acc[k + 1];
        acc[WZ - 1].x = (T)0; acc[WZ - 1].y = (T)0;
    }
}

}  // namespace enuf
