// Step a2 -- spreading (adjoint NFFT, part 1):
//   g[l] = sum_j q_j phi(u_jx - l_x) phi(u_jy - l_y) phi(u_jz - l_z), l periodic.
//
// Output-stationary, sliding z-window, warp-specialised.  The work is the set of SLABS (column, bin plane): a column
// is CX x 16 grid cells in (x, y) (CX = 32, or 16 on small grids), slab s of a column holds the particles binned to
// plane s, whose stencils reach the planes s - SHI .. s + SLO.  The ncol * n slabs are cut into PIECES (column, [z0, z1))
// and shared equally among as many CTAs as the device holds at once (SpreadSplit, enuf_common.cuh: most CTAs get one
// piece, cut at the same planes in every column; the rest share the columns' remainders).  A CTA stages every slab of
// its pieces exactly once -- there is no halo in z: the
// WZ - 1 planes at either end of a piece, which also receive from the neighbouring piece, are added into the grid
// with red.global.add (those planes of the column are zeroed beforehand by spread_zero_block, run as extra blocks of
// the first kernel of the evaluation; each such value is 0 + a + b with a, b the two pieces' sums, so the result does
// not depend on the order), all other planes are complete and written with one plain store.  A CTA has
//   - NCONS = CX/8 x 2 CONSUMER warps, each owning an 8 x 8 patch of the column: every lane owns two
//     x-adjacent cells and keeps, in registers, their partial sums on the WZ consecutive planes that the
//     particles of slab s (bin plane s) can reach.  Per (warp, particle) visit the work is WZ packed FMAs
//     acc[k] += (a0, a1) * (q wz[k]) with (a0, a1) = wx[cells] * wy[cell].  After slab s the lowest plane
//     of the window has everything this piece sends to it: one coalesced store (or reduction, see above), and the
//     window slides.  No shared-memory read-modify-write, no clearing of the whole grid;
//   - four PRODUCER warps taking the slabs in turn (slab i of the chunk goes to stage i % 3 of a three-stage ring):
//     a producer culls the particles of the neighbouring bins against the column's halo, copies the three
//     window rows of the accepted ones (evaluated ONCE per particle by window_rows_kernel, enuf_bin.cuh --
//     "window values computed [once and kept]") into slots of its stage with cp.async, builds
//     for every patch the list of staged particles whose stencil overlaps it, and hands the stage over
//     through mbarriers (full / empty / again per producer; the copies arrive on the full barrier themselves).
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
// kSparse: few particles per slab and column (the plan decides, enuf_api.cu): rounds of 32 slots in an eight-stage ring
// instead of 96 in three -- the same shared memory, but the flight time of the row copies after a hand-over (which is
// what bounds a sparse slab) is spread over eight slabs.  Correct for any density (a denser slab takes several rounds).
template <typename T, int M_, bool kTrim, int NPX_, bool kSparse = false>
struct SpreadCfg {
    static constexpr int W = 2 * M_ + 1;
    static constexpr int WZ = W - (kTrim ? 1 : 0);               // stencil points per dimension = planes in the window
    static constexpr int SLO = M_, SHI = kTrim ? M_ - 1 : M_;    // slab s reaches the planes s - SHI .. s + SLO
    static constexpr int NPX = NPX_, NPY = 2, NCONS = NPX * NPY; // 8 x 8 patches = consumer warps
    static constexpr int NPROD = 4;                              // producer warps: producer k takes the slabs k, k + 4, .. of the chunk
    static constexpr int NSTAGE = kSparse ? 8 : 3;               //   slab i of the chunk is staged in stage i % NSTAGE
    static constexpr int CX = 8 * NPX, CY = 8 * NPY;             // column
    static constexpr int NT = 32 * (NCONS + NPROD);
    static constexpr int NBX = CX / kTile + 2, NBY = CY / kTile + 2;   // bins (16 x 16, enuf_common.cuh) the halo touches
    static constexpr int NSEG = 2 * NBY;                         // ranges of the sorted array per slab (<= 2 per row of bin columns)
    // slot layout (elements of T): zeros | x row | zeros | y row | zeros | z row ; the largest index a lane reads is
    // x: 8 + 1 + (WZ-1) + 7, y: OYF + (WZ-1) + 7 (header comment)
    static constexpr int OXF = 8;
    static constexpr int OYF = (16 + WZ + 3) / 4 * 4 > 24 ? (16 + WZ + 3) / 4 * 4 : 24;
    static constexpr int OZF = (OYF + WZ + 7 + 3) / 4 * 4 > OYF + 16 ? (OYF + WZ + 7 + 3) / 4 * 4 : OYF + 16;
    static constexpr int PITCH = OZF + 16 <= 68 ? 68 : 76;       // = 4 / 12 mod 32: 16-byte row chunks of 8 slots hit 32 banks
    static constexpr int CAP = kSparse ? 32 :
        (sizeof(T) == 4 ? (NPX == 4 ? (PITCH == 68 ? 96 : 88) : 56) : (NPX == 4 ? 48 : 40));   // staged particles per round
    static constexpr int LCAP = CAP + 4;                         // visit-list entries per patch (even padding + prefetch)
    static constexpr int kBlk = 16;                              // slabs (of one producer) whose bin ranges are loaded at once
    static constexpr int CTAS_PER_SM = sizeof(T) == 4 ? (NPX == 4 ? 2 : 3) : (NPX == 4 ? 1 : 2);
    static constexpr size_t SLOT_BYTES = sizeof(T) * (size_t)(CAP + 1) * PITCH;   // slot CAP is all zero
    static constexpr size_t LIST_BYTES = sizeof(uint2) * (size_t)NCONS * LCAP;
    static constexpr size_t STAGE_BYTES = ((SLOT_BYTES + LIST_BYTES + 15) / 16) * 16;
    static_assert(CAP >= 32 && CAP + 1 < 256 && NCONS <= 8, "a cull step stages up to 32 particles; packed list lengths");
    static_assert(NSEG <= 8 && kBlk == 16, "segment table: 8 packed ends + 8 offsets per slab; lanes = 16 slabs x (start, end)");
    static_assert(NPROD == 4, "barrier protocol: slab i - NSTAGE held the stage, its producer is (k - NSTAGE) & 3");
    // A barrier may run at most one phase ahead of its waiter.  With full / empty barriers per PRODUCER that holds as
    // long as NSTAGE <= NPROD (slab i + 4 can be staged / finished only after slab i was consumed / its stage re-staged);
    // the eight-stage ring keeps them per STAGE instead, where it holds for any depth.
    static constexpr bool kStageBars = NSTAGE > NPROD;
    static constexpr int NBAR = kStageBars ? NSTAGE : NPROD;
    static_assert(SLOT_BYTES < 65536, "visit-list entries are 16-bit byte offsets");
    static_assert(OZF + 16 <= PITCH, "slot layout");
};

template <typename T, int M_, bool kTrim, int NPX, bool kSparse = false>
constexpr size_t spread_smem_bytes() {
    using C = SpreadCfg<T, M_, kTrim, NPX, kSparse>;
    return C::STAGE_BYTES * C::NSTAGE;
}

// The three window rows of one particle, as the spreading kernel stages them (evaluated once per particle by
// window_rows_kernel, enuf_bin.cuh, read by every CTA whose halo the particle is in): RP elements per particle,
//   x row [0, 16):        element j = phi_x at stencil point j - parx (parx = parity of the first stencil point's grid index),
//   y row [16, 16 + RY):  element j = phi_y at stencil point j,
//   z row [16 + RY, RP):  element j = q phi_z at stencil point j,
// zero beyond the WZ stencil points.  kTrim: stencil point k is point k + ks of the 2m+1 (ks = d0 > 0).
template <int M_, bool kTrim>
struct WindowRows {
    static constexpr int W = 2 * M_ + 1, WZ = W - (kTrim ? 1 : 0);
    static constexpr int RX = 16, RY = (WZ + 3) / 4 * 4, OY = RX, OZ = RX + RY, RP = RX + 2 * RY;
    static_assert(WZ + 1 <= RX, "x row: WZ points + one parity element");
};

template <typename T, int M_, bool kTrim>
__device__ __forceinline__ void write_window_row(const WindowParams& wp, const PolyArg<M_>& pa, int dim, T d0, T q,
                                                 int parx, T* __restrict__ dst) {
    using R = WindowRows<M_, kTrim>;
    constexpr int W = R::W, WZ = R::WZ;
    using V4 = typename Vec4<T>::type;
    T w[W], dw[W];
    stencil_weights<T, M_, false>(wp, pa, d0, w, dw);
    const int sh = (kTrim && d0 > (T)0) ? 1 : 0;
    const int par = dim == 0 ? parx : 0;
    const T mult = dim == 2 ? q : (T)1;
    constexpr int RMAX = R::RX;
    T rr[RMAX];
#pragma unroll
    for (int j = 0; j < RMAX; ++j) {
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
        rr[j] = v * mult;
    }
    const int len = dim == 0 ? R::RX : R::RY;
    V4* row4 = reinterpret_cast<V4*>(dst + (dim == 0 ? 0 : (dim == 1 ? R::OY : R::OZ)));
#pragma unroll
    for (int v = 0; v < RMAX / 4; ++v) {
        if (4 * v < len) {
            V4 o; o.x = rr[4 * v]; o.y = rr[4 * v + 1]; o.z = rr[4 * v + 2]; o.w = rr[4 * v + 3];
            row4[v] = o;
        }
    }
}

// The grid planes that two pieces share are zeroed before the spreading kernel adds into them: block i of G + ncol clears
// the `nzp` = WZ - 1 planes from z0 - shi on (mod n) of the column where piece start i lies (spread_piece_start,
// enuf_common.cuh).  Run as extra blocks of bin_count_kernel.
template <typename T>
struct SpreadZero {
    T* grid;            // nullptr: nothing to do
    SpreadSplit sp;
    int cx, cy;         // column footprint
    int shi, nzp;       // planes z0 - shi .. z0 - shi + nzp - 1
};
template <typename T>
__device__ __forceinline__ void spread_zero_block(const SpreadZero<T>& zr, int i) {
    const SpreadSplit& sp = zr.sp;
    int col, z0;
    if (!spread_piece_start(sp, i, col, z0)) return;
    const int ncolx = sp.n / zr.cx, Tx = col % ncolx, Ty = col / ncolx;
    constexpr int VE = 16 / (int)sizeof(T);                 // elements per 16-byte store
    const int vx = zr.cx / VE, per_plane = zr.cy * vx;
    const uint4 zero = make_uint4(0u, 0u, 0u, 0u);
    for (int e = threadIdx.x; e < zr.nzp * per_plane; e += blockDim.x) {
        const int k = e / per_plane, rem = e - k * per_plane, y = rem / vx, xv = rem - y * vx;
        int pz = z0 - zr.shi + k;
        pz += pz < 0 ? sp.n : 0; pz -= pz >= sp.n ? sp.n : 0;
        T* dst = zr.grid + ((size_t)pz * sp.n + (size_t)(Ty * zr.cy + y)) * sp.n + Tx * zr.cx + xv * VE;
        *reinterpret_cast<uint4*>(dst) = zero;
    }
}

// grid[addr] += v for a pair of x-adjacent cells, without a return value (L2 reduction)
__device__ __forceinline__ void red_pair(float2* addr, const float2 v) {
    asm volatile("red.global.add.v2.f32 [%0], {%1, %2};" ::"l"(addr), "f"(v.x), "f"(v.y) : "memory");
}
__device__ __forceinline__ void red_pair(double2* addr, const double2 v) {
    asm volatile("red.global.add.f64 [%0], %1;" ::"l"(addr), "d"(v.x) : "memory");
    asm volatile("red.global.add.f64 [%0], %1;" ::"l"(reinterpret_cast<double*>(addr) + 1), "d"(v.y) : "memory");
}

// explicit shared-space loads (32-bit shared addresses: no generic-to-shared conversion inside the visit loop)
template <typename T> __device__ __forceinline__ typename Pair2<T>::type lds_pair(uint32_t a);
template <> __device__ __forceinline__ float2 lds_pair<float>(uint32_t a) {
    float2 v; asm volatile("ld.shared.v2.f32 {%0, %1}, [%2];" : "=f"(v.x), "=f"(v.y) : "r"(a)); return v;
}
template <> __device__ __forceinline__ double2 lds_pair<double>(uint32_t a) {
    double2 v; asm volatile("ld.shared.v2.f64 {%0, %1}, [%2];" : "=d"(v.x), "=d"(v.y) : "r"(a)); return v;
}
template <typename T> __device__ __forceinline__ T lds_one(uint32_t a);
template <> __device__ __forceinline__ float lds_one<float>(uint32_t a) {
    float v; asm volatile("ld.shared.f32 %0, [%1];" : "=f"(v) : "r"(a)); return v;
}
template <> __device__ __forceinline__ double lds_one<double>(uint32_t a) {
    double v; asm volatile("ld.shared.f64 %0, [%1];" : "=d"(v) : "r"(a)); return v;
}
template <typename T> __device__ __forceinline__ typename Vec4<T>::type lds_quad(uint32_t a);
template <> __device__ __forceinline__ float4 lds_quad<float>(uint32_t a) {
    float4 v; asm volatile("ld.shared.v4.f32 {%0, %1, %2, %3}, [%4];" : "=f"(v.x), "=f"(v.y), "=f"(v.z), "=f"(v.w) : "r"(a)); return v;
}
template <> __device__ __forceinline__ double4 lds_quad<double>(uint32_t a) {
    double4 v;
    asm volatile("ld.shared.v2.f64 {%0, %1}, [%2];" : "=d"(v.x), "=d"(v.y) : "r"(a));
    asm volatile("ld.shared.v2.f64 {%0, %1}, [%2];" : "=d"(v.z), "=d"(v.w) : "r"(a + 16u));
    return v;
}
__device__ __forceinline__ int lds_s32(uint32_t a) {
    int v;
    asm volatile("ld.shared.s32 %0, [%1];" : "=r"(v) : "r"(a));
    return v;
}
__device__ __forceinline__ uint2 lds_u2(uint32_t a) {
    uint2 v; asm volatile("ld.shared.v2.u32 {%0, %1}, [%2];" : "=r"(v.x), "=r"(v.y) : "r"(a)); return v;
}

__device__ __forceinline__ void cp_async_16(uint32_t smem_dst, const void* gmem_src) {
    asm volatile("cp.async.cg.shared.global [%0], [%1], 16;" ::"r"(smem_dst), "l"(gmem_src) : "memory");
}
// the mbarrier receives one arrival when all cp.async operations this thread has issued so far are complete
__device__ __forceinline__ void cp_async_mbar_arrive(uint64_t* bar) {
    asm volatile("cp.async.mbarrier.arrive.noinc.shared::cta.b64 [%0];" ::"r"(smem_u32(bar)) : "memory");
}

// slots[].cell: bits 0..29 the packed nearest cell, bits 30 / 31 = ks_x / ks_y (trimmed plans; enuf_bin.cuh)
// rows: [N][RP] window rows in bin order (WindowRows)
template <typename T, int M_, bool kTrim, int NPX, bool kSparse = false>
__global__ void __launch_bounds__((SpreadCfg<T, M_, kTrim, NPX, kSparse>::NT), (SpreadCfg<T, M_, kTrim, NPX, kSparse>::CTAS_PER_SM))
spread_kernel(const PSlot<T>* __restrict__ slots, const T* __restrict__ rows,
              const uint32_t* __restrict__ offset, TileGeom g, SpreadSplit sp, T* __restrict__ grid) {
    pdl_prologue();
    SpreadPiece pc;
    if (!spread_piece(sp, (int)blockIdx.x, 0, pc)) return;  // (an empty range: its boundaries were moved onto each other)
    using C = SpreadCfg<T, M_, kTrim, NPX, kSparse>;
    using R = WindowRows<M_, kTrim>;
    using P2 = typename Pair2<T>::type;
    using V4 = typename Vec4<T>::type;
    constexpr int WZ = C::WZ, NCONS = C::NCONS, CX = C::CX, CY = C::CY, CAP = C::CAP, LCAP = C::LCAP;
    constexpr int PITCH = C::PITCH, OXF = C::OXF, OYF = C::OYF, OZF = C::OZF;
    constexpr int NSTAGE = C::NSTAGE, kBlk = C::kBlk, NSEG = C::NSEG;
    constexpr unsigned ES = (unsigned)sizeof(T);
    constexpr unsigned FULL = 0xffffffffu;

    extern __shared__ __align__(16) unsigned char smem_raw[];
    // per producer k: full_bar[k]  -- a round of one of its slabs is staged (consumers wait),
    //                 again_bar[k] -- every consumer is done with a round that was not the slab's last (producer k waits),
    //                 empty_bar[k] -- every consumer is done with the last round of a slab of producer k: its stage is
    //                                 free for the slab NSTAGE further on, i.e. for producer (k + NSTAGE) & 3 (only that one waits on it).
    // Every barrier has one waiting party that sees each of its phases in turn, so one parity bit per party suffices.
    // (kStageBars: full_bar / empty_bar are indexed by the stage instead, the phases of empty_bar[stage] are the slabs
    //  stage, stage + NSTAGE, .. of the chunk, so the waiter's parity follows from the slab index.)
    __shared__ uint64_t full_bar[C::NBAR], empty_bar[C::NBAR], again_bar[C::NPROD];
    __shared__ int cl_s[NSTAGE][NCONS];         // visits of each patch in the stage | 0x10000 if it is the slab's last round
    // candidates of a slab = its NSEG ranges of the sorted array laid end to end ("packed" numbering e = 0 .. total - 1);
    // per slab: [0..6] packed end of segment 0..6 (total from segment NSEG - 1 on), [7] total, [8 + i] = start of
    // segment i - its packed start, so that candidate e of segment i is slots[e + [8 + i]]
    __shared__ __align__(16) uint32_t segtab[C::NPROD][kBlk][16];
    __shared__ uint2 acc_rec[C::NPROD][CAP];            // producer's side buffer: accepted particles of the round,
                                                        //   (sorted-array index, (X0 + 32) | (Y0 + 32) << 8)

    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int ncolx = g.n / CX;

    // the zero padding of every slot (and the all-zero slot CAP) is written once; rows are rewritten per round
    for (int i = tid; i < (int)(C::STAGE_BYTES * NSTAGE / 16); i += C::NT)
        reinterpret_cast<uint4*>(smem_raw)[i] = make_uint4(0u, 0u, 0u, 0u);
    if (tid == 0) {
#pragma unroll
        for (int st = 0; st < C::NBAR; ++st) {
            // full: one arrival per producer lane when its row copies have landed + one after the lists are written
            mbar_init(&full_bar[st], 33);
            mbar_init(&empty_bar[st], NCONS);
        }
#pragma unroll
        for (int st = 0; st < C::NPROD; ++st) mbar_init(&again_bar[st], NCONS);
    }
    __syncthreads();

    if (warp >= NCONS) {
        // =========================================================== producers
        // the slabs of the CTA's pieces are numbered gi = 0, 1, .. in the order they are worked through; producer k stages
        // the slabs gi = k, k + 4, ..; slab gi goes to stage gi % NSTAGE
        const int k = warp - NCONS;
        const int half = lane >> 4, l16 = lane & 15;
        const unsigned below = (1u << lane) - 1u;
        const uint4* tb = reinterpret_cast<const uint4*>(segtab[k]);
        unsigned pe = 0, pa = 0;                 // parities of the next phase of empty_bar[(k - NSTAGE) & 3] / again_bar[k] to wait for
        // per piece (set in the loop over pieces below): the halo's segments, the cull offsets, the block of loaded ranges
        int seg_bin0 = 0, seg_nb = 0, offx = 0, offy = 0, blk0 = 0;
        // candidates of a slab, 32 per step, in packed numbering (segtab): a sparse slab is ONE step however its
        // particles are spread over the segments.  The cell words of up to kSteps steps are loaded together (one
        // global-load latency per slab, not one per step), then examined in order; those of the producer's NEXT slab
        // are started as soon as the current slab is culled, so that they arrive during the hand-over, the lists and
        // the copies.
        constexpr int kSteps = 8;
        uint32_t ebase = 0, total = 0;           // first candidate of the next load, candidates of the slab
        uint32_t cw[kSteps], cidx[kSteps];
        int nst = 0;                             // steps loaded (consumed ones are marked invalid)
        bool preloaded = false;                  // cw / cidx already hold the first steps of this slab
        auto load_steps = [&](int js) {
            const uint4 e0 = tb[4 * js], e1 = tb[4 * js + 1], d0 = tb[4 * js + 2], d1 = tb[4 * js + 3];
            const uint32_t pe_[7] = {e0.x, e0.y, e0.z, e0.w, e1.x, e1.y, e1.z};
            const uint32_t dl_[8] = {d0.x, d0.y, d0.z, d0.w, d1.x, d1.y, d1.z, d1.w};
            total = e1.w;
            nst = 0;
#pragma unroll
            for (int j = 0; j < kSteps; ++j) {
                cw[j] = 0xffffffffu;
                cidx[j] = 0u;
                if (ebase + 32u * j < total) {
                    const uint32_t e = ebase + 32u * j + (uint32_t)lane;
                    uint32_t dl = dl_[0];
#pragma unroll
                    for (int i = 0; i + 1 < NSEG; ++i) dl = e >= pe_[i] ? dl_[i + 1] : dl;
                    cidx[j] = e + dl;
                    if (e < total) cw[j] = slots[cidx[j]].cell;
                    nst = j + 1;
                }
            }
            ebase += 32u * kSteps;
        };
        int gs = 0;                              // number of the piece's first slab
        for (int pi = 0; spread_piece(sp, (int)blockIdx.x, pi, pc); ++pi) {
        const int z0 = pc.z0, z1 = pc.z1;
        const int Tx = pc.col % ncolx, Ty = pc.col / ncolx;
        // The halo of the column touches NBY rows of NBX bin columns; in bin order (TileGeom) the NBX bins of one
        // row and plane are adjacent, so a slab is NBY ranges of the sorted array, each split in two where the
        // row of columns wraps around the box (segments 2 jy, 2 jy + 1).  Lane sg < NSEG: (first bin of plane 0,
        // number of bins) of segment sg.  Rows / columns the periodic box holds only once are taken once.
        seg_bin0 = 0; seg_nb = 0;
        if (lane < NSEG) {
            const int jy = lane >> 1, second = lane & 1;
            const int nrow = C::NBY < g.nt ? C::NBY : g.nt, nbx = C::NBX < g.nt ? C::NBX : g.nt;
            int ty = Ty * (CY / kTile) - 1 + jy;
            ty += ty < 0 ? g.nt : 0; ty -= ty >= g.nt ? g.nt : 0;
            int txlo = Tx * (CX / kTile) - 1;
            txlo += txlo < 0 ? g.nt : 0;
            if (nbx == g.nt) txlo = 0;
            const int na = min(nbx, g.nt - txlo);        // bins before the wrap
            const int tx = second ? 0 : txlo;
            seg_nb = jy < nrow ? (second ? nbx - na : na) : 0;
            seg_bin0 = bin_index(g, tx, ty, 0);
        }
        // first stencil point in column coordinates from the packed cell: the periodic image that can overlap the column
        offx = -M_ - CX * Tx + (WZ - 1); offy = -M_ - CY * Ty + (WZ - 1);
        const int s_first = z0 + ((k - gs) & 3);  // this producer's first slab of the piece
        blk0 = s_first - C::NPROD * kBlk;
        preloaded = false;
        for (int s = s_first; s < z1; s += C::NPROD) {
            const int gi = gs + (s - z0);
            if (s - blk0 >= C::NPROD * kBlk) {
                // ranges of this producer's next kBlk slabs: lane & 15 = slab, lanes 0..15 load the starts, 16..31 the ends
                blk0 = s;
                __syncwarp();
                const int cz = (blk0 + C::NPROD * l16) % g.n;              // (slabs past the piece's end are loaded but not used)
                uint32_t pend[8], pdel[8], run = 0u;
#pragma unroll
                for (int sg = 0; sg < 8; ++sg) { pend[sg] = 0u; pdel[sg] = 0u; }
#pragma unroll
                for (int sg = 0; sg < NSEG; ++sg) {
                    const int b0 = __shfl_sync(FULL, seg_bin0, sg), nb = __shfl_sync(FULL, seg_nb, sg);
                    const uint32_t v = offset[b0 + cz * g.nt + half * nb];
                    const uint32_t ve = __shfl_down_sync(FULL, v, 16);      // lanes < 16: the end of the range
                    pdel[sg] = v - run;
                    run += ve - v;
                    pend[sg] = run;
                }
#pragma unroll
                for (int sg = NSEG - 1; sg < 8; ++sg) pend[sg] = run;       // [NSEG - 1 .. 7] = total
                if (lane < kBlk) {
                    uint4* t4 = reinterpret_cast<uint4*>(segtab[k][lane]);
                    t4[0] = make_uint4(pend[0], pend[1], pend[2], pend[3]);
                    t4[1] = make_uint4(pend[4], pend[5], pend[6], pend[7]);
                    t4[2] = make_uint4(pdel[0], pdel[1], pdel[2], pdel[3]);
                    t4[3] = make_uint4(pdel[4], pdel[5], pdel[6], pdel[7]);
                }
                __syncwarp();
            }
            const int js = (s - blk0) / C::NPROD;
            const int stage = gi % NSTAGE;
            unsigned char* sbase = smem_raw + (size_t)stage * C::STAGE_BYTES;
            const uint32_t sl32 = smem_u32(sbase);
            uint2* lists = reinterpret_cast<uint2*>(sbase + C::SLOT_BYTES);
            if (!preloaded) { ebase = 0u; load_steps(js); }
            preloaded = false;
            bool slab_done = false, first_round = true;
            while (!slab_done) {
                // ---- cull (before the stage is free: it needs only this producer's side buffer): accepted particles'
                //      sorted-array index and packed stencil origin; their rows are started towards L2
                int ns = 0;
                for (;;) {
                    // all loaded steps at once (the steps are independent up to the running slot count)
                    int pkv[kSteps]; unsigned bal[kSteps];
#pragma unroll
                    for (int j = 0; j < kSteps; ++j) { pkv[j] = -1; bal[j] = 0u; }
#pragma unroll
                    for (int j = 0; j < kSteps; ++j) {
                        if (j < nst) {                                  // (uniform)
                            const uint32_t cwj = cw[j];
                            // (c + ks + off lies in (-n, 2n): wrapped into [0, n) without assuming a power of two)
                            int vx = (int)(cwj & 1023u) + (int)((cwj >> 30) & 1u) + offx;
                            int vy = (int)((cwj >> 10) & 1023u) + (int)(cwj >> 31) + offy;
                            vx += vx < 0 ? g.n : 0; vx -= vx >= g.n ? g.n : 0;
                            vy += vy < 0 ? g.n : 0; vy -= vy >= g.n ? g.n : 0;
                            const int X0 = vx - (WZ - 1), Y0 = vy - (WZ - 1);
                            const bool ok = cwj != 0xffffffffu && X0 <= CX - 1 && Y0 <= CY - 1;
                            bal[j] = __ballot_sync(FULL, ok);
                            pkv[j] = ok ? ((X0 + 32) | ((Y0 + 32) << 8)) : -1;
                        }
                    }
                    // steps are taken while their accepted particles fit into the round (CAP slots)
                    int jl = kSteps, base = ns, pb[kSteps];
#pragma unroll
                    for (int j = 0; j < kSteps; ++j) {
                        const int c = __popc(bal[j]);
                        if (jl == kSteps && base + c > CAP) jl = j;
                        pb[j] = base;
                        if (j < jl) base += c;
                    }
#pragma unroll
                    for (int j = 0; j < kSteps; ++j) {
                        if (j < nst && j < jl) {
                            if (pkv[j] >= 0)
                                acc_rec[k][pb[j] + __popc(bal[j] & below)] = make_uint2(cidx[j], (unsigned)pkv[j]);
                            cw[j] = 0xffffffffu;                        // consumed
                        }
                    }
                    ns = base;
                    if (jl < kSteps) break;                            // step jl opens the next round of this slab
                    if (ebase >= total) { slab_done = true; break; }   // the ranges are exhausted
                    load_steps(js);                                    // a long slab: the next kSteps steps
                }
                if (slab_done && s + C::NPROD < z1 && js + 1 < kBlk) {
                    ebase = 0u;
                    load_steps(js + 1);                                // the next slab of this producer (same block of ranges)
                    preloaded = true;
                }
                __syncwarp();
                // ---- visit lists, first half (still before the hand-over): for every patch the staged particles whose
                //      stencil overlaps it (ballot + popc compaction), kept in registers -- per group of 32 slots the patch
                //      mask, the 8 list positions (bytes of two words) and the ready-made byte offsets of the x and y rows.
                //      (A round stages at most CAP + 1 < 256 entries per list, so list lengths are bytes of lcp[].)
                constexpr int NGRP = (CAP + 31) / 32;
                unsigned lcp[2] = {0u, 0u}, lmask[NGRP], lpos[NGRP][2], lxb[NGRP], lyb[NGRP];
#pragma unroll
                for (int gq = 0; gq < NGRP; ++gq) {
                    lmask[gq] = 0u; lpos[gq][0] = lpos[gq][1] = 0u; lxb[gq] = lyb[gq] = 0u;
                    if (32 * gq < ns) {
                        const int slot = 32 * gq + lane;
                        const bool v = slot < ns;
                        int X0 = 64, Y0 = 64;
                        if (v) { const int pkv = (int)acc_rec[k][slot].y; X0 = (pkv & 255) - 32; Y0 = ((pkv >> 8) & 255) - 32; }
                        const unsigned sb = (unsigned)(slot * PITCH) * ES;
                        lxb[gq] = sb + (unsigned)(OXF + (X0 & 1) - X0) * ES;
                        lyb[gq] = sb + (unsigned)(OYF - Y0) * ES;
#pragma unroll
                        for (int w8 = 0; w8 < NCONS; ++w8) {
                            const int px0 = 8 * (w8 % NPX), py0 = 8 * (w8 / NPX);
                            const bool ov = v && X0 <= px0 + 7 && X0 + WZ - 1 >= px0 && Y0 <= py0 + 7 && Y0 + WZ - 1 >= py0;
                            const unsigned bal = __ballot_sync(FULL, ov);
                            const unsigned cur = (lcp[w8 >> 2] >> (8 * (w8 & 3))) & 255u;
                            lmask[gq] |= ov ? (1u << w8) : 0u;
                            lpos[gq][w8 >> 2] |= (cur + (unsigned)__popc(bal & below)) << (8 * (w8 & 3));
                            lcp[w8 >> 2] += (unsigned)__popc(bal) << (8 * (w8 & 3));
                        }
                    }
                }
                if (first_round) {
                    // the slab that held the stage before (s - NSTAGE, staged by producer (k - NSTAGE) & 3) must be finished
                    if (gi >= NSTAGE) {
                        if constexpr (C::kStageBars) {
                            mbar_wait_backoff(&empty_bar[stage], (unsigned)((gi / NSTAGE - 1) & 1));
                        } else {
                            mbar_wait_backoff(&empty_bar[(k - NSTAGE) & 3], pe); pe ^= 1u;
                        }
                    }
                    first_round = false;
                } else {
                    mbar_wait_backoff(&again_bar[k], pa); pa ^= 1u;     // the previous round of this slab
                }
                __syncwarp();
                // ---- visit lists, second half: the entries worked out before the hand-over are stored into the stage
#pragma unroll
                for (int gq = 0; gq < NGRP; ++gq) {
                    if (32 * gq < ns) {
                        const unsigned zb = (unsigned)((32 * gq + lane) * PITCH + OZF) * ES;
#pragma unroll
                        for (int w8 = 0; w8 < NCONS; ++w8) {
                            const int px0 = 8 * (w8 % NPX), py0 = 8 * (w8 / NPX);
                            if ((lmask[gq] >> w8) & 1u)
                                lists[w8 * LCAP + ((lpos[gq][w8 >> 2] >> (8 * (w8 & 3))) & 255u)] =
                                    make_uint2((lxb[gq] + (unsigned)px0 * ES) | (zb << 16), lyb[gq] + (unsigned)py0 * ES);
                        }
                    }
                }
                if (lane < NCONS) {                                        // lane w8 closes list w8
                    const unsigned zs = (unsigned)(CAP * PITCH) * ES;      // the all-zero slot
                    const int c = (int)(((lane < 4 ? lcp[0] : lcp[1]) >> (8 * (lane & 3))) & 255u);
                    // even length, and the consumer loads its operands one visit ahead: entries that point at the zero slot
                    lists[lane * LCAP + c] = lists[lane * LCAP + c + 1] = lists[lane * LCAP + c + 2] =
                        make_uint2((zs + OXF * ES) | ((zs + OZF * ES) << 16), zs + OYF * ES);
                    cl_s[stage][lane] = (c + (c & 1)) | (slab_done ? 0x10000 : 0);
                }
                // ---- copy the window rows of the accepted particles into the slots (cp.async; they arrive on full_bar themselves)
                for (int g0 = 0; g0 < ns; g0 += 32) {
                    const int pos = g0 + lane;
                    if (pos < ns) {
                        const char* src = reinterpret_cast<const char*>(rows + (size_t)acc_rec[k][pos].x * R::RP);
                        const uint32_t dst = sl32 + (uint32_t)(pos * PITCH) * ES;
                        constexpr int CHX = (int)(R::RX * sizeof(T) / 16), CHY = (int)(R::RY * sizeof(T) / 16);
#pragma unroll
                        for (int c = 0; c < CHX; ++c) cp_async_16(dst + OXF * ES + 16 * c, src + 16 * c);
#pragma unroll
                        for (int c = 0; c < CHY; ++c) cp_async_16(dst + OYF * ES + 16 * c, src + R::OY * ES + 16 * c);
#pragma unroll
                        for (int c = 0; c < CHY; ++c) cp_async_16(dst + OZF * ES + 16 * c, src + R::OZ * ES + 16 * c);
                    }
                }
                uint64_t* fb = &full_bar[C::kStageBars ? stage : k];
                cp_async_mbar_arrive(fb);
                __syncwarp();                                       // lane 0's arrive (release) publishes every lane's list entries
                if (lane == 0) mbar_arrive(fb);
            }
        }
        gs += z1 - z0;
        }
        return;
    }

    // =============================================================== consumers
    const int px0 = 8 * (warp % NPX), py0 = 8 * (warp / NPX);
    const int lxl = (lane & 3) * 2, lyl = lane >> 2;              // this lane's two cells (lxl, lyl), (lxl + 1, lyl) of the patch
    const size_t plane = (size_t)g.n * g.n;
    constexpr int NV = (WZ + 3) / 4;

    P2 acc[WZ];
#pragma unroll
    for (int kk = 0; kk < WZ; ++kk) { acc[kk].x = (T)0; acc[kk].y = (T)0; }

    // operands of one visit: this lane's (wx pair, wy) and the particle's q * z row
    struct Ops { P2 wx; T wy; V4 z[NV]; };
    auto load_ops = [&](uint32_t sbx, uint32_t sby, uint32_t sbz, uint2 e) {
        Ops o;
        o.wx = lds_pair<T>(sbx + (e.x & 0xffffu));
        o.wy = lds_one<T>(sby + e.y);
        const uint32_t za = sbz + (e.x >> 16);
#pragma unroll
        for (int v = 0; v < NV; ++v) o.z[v] = lds_quad<T>(za + v * (uint32_t)sizeof(V4));
        return o;
    };

    unsigned pf = 0;                                              // parity bits of the next phase of full_bar[..]
    // everything a slab needs is kept as a shared-window address or stepped along, so that an empty slab costs a
    // wait, one load, one arrive, the store and the slide (dilute systems are bound by exactly that)
    const uint32_t smem32 = smem_u32(smem_raw);
    const uint32_t fb32 = smem_u32(full_bar), eb32 = smem_u32(empty_bar), ab32 = smem_u32(again_bar);
    const uint32_t cl32 = smem_u32(cl_s) + (uint32_t)warp * 4u;
    const uint32_t lpw = (uint32_t)C::SLOT_BYTES + (uint32_t)(warp * LCAP * sizeof(uint2));
    int stage = 0, prod = 0;
    for (int pi = 0; spread_piece(sp, (int)blockIdx.x, pi, pc); ++pi) {
    const int z0 = pc.z0, z1 = pc.z1;
    const int Tx = pc.col % ncolx, Ty = pc.col / ncolx;
    T* gcol = grid + ((size_t)(Ty * CY + py0 + lyl)) * g.n + Tx * CX + px0 + lxl;     // this lane's cells on plane 0
    int pz = z0 - C::SHI;                                       // plane the next slab completes (mod n)
    pz += pz < 0 ? g.n : 0;
    for (int s = z0; s < z1; ++s) {
        const int bar = C::kStageBars ? stage : prod;
        const uint32_t sbz = smem32 + (uint32_t)stage * (uint32_t)C::STAGE_BYTES;
        const uint32_t sbx = sbz + lxl * ES, sby = sbz + lyl * ES;
        const uint32_t lp = sbz + lpw;
        int cl;
        do {
            mbar_wait_backoff(fb32 + 8u * (uint32_t)bar, (pf >> bar) & 1u);
            pf ^= 1u << bar;
            cl = lds_s32(cl32 + (uint32_t)stage * (uint32_t)(NCONS * 4));
            const int cnt = cl & 0xffff;
            // one visit ahead: while visit i is accumulated, the operands of visit i + 1 and the entry of visit i + 2 are
            // in flight.  Two visits per trip (A, B alternate, no register moves); the list is padded with entries that
            // point at the all-zero slot: to an even length, and two more for the loads that run ahead.
            if (cnt > 0) {                                          // (sparse systems: most patches see no particle in a slab)
                Ops A = load_ops(sbx, sby, sbz, lds_u2(lp));
                uint2 en = lds_u2(lp + 8);
                for (int i = 0; i < cnt; i += 2) {
                    const Ops B = load_ops(sbx, sby, sbz, en);
                    en = lds_u2(lp + 8 * (uint32_t)(i + 2));
                    {
                        const P2 a = pair_scale(A.wx, A.wy);
                        const T* wz = reinterpret_cast<const T*>(A.z);
#pragma unroll
                        for (int kk = 0; kk < WZ; ++kk) fma_pair(acc[kk], a, wz[kk]);
                    }
                    A = load_ops(sbx, sby, sbz, en);
                    en = lds_u2(lp + 8 * (uint32_t)(i + 3));
                    {
                        const P2 a = pair_scale(B.wx, B.wy);
                        const T* wz = reinterpret_cast<const T*>(B.z);
#pragma unroll
                        for (int kk = 0; kk < WZ; ++kk) fma_pair(acc[kk], a, wz[kk]);
                    }
                }
            }
            __syncwarp();
            if (lane == 0) mbar_arrive((cl >> 16) ? eb32 + 8u * (uint32_t)bar : ab32 + 8u * (uint32_t)prod);
        } while (!(cl >> 16));
        // the lowest plane of the window, s - SHI, has received everything this piece sends to it.  It is complete
        // (plain store) unless it is one of the piece's first WZ - 1 planes, which the piece below also adds to
        {
            P2* out = reinterpret_cast<P2*>(gcol + (size_t)pz * plane);
            if (s - z0 >= WZ - 1) *out = acc[0];
            else red_pair(out, acc[0]);
        }
        pz = pz + 1 == g.n ? 0 : pz + 1;
#pragma unroll
        for (int kk = 0; kk + 1 < WZ; ++kk) acc[kk] = acc[kk + 1];
        acc[WZ - 1].x = (T)0; acc[WZ - 1].y = (T)0;
        stage = stage + 1 == NSTAGE ? 0 : stage + 1;
        prod = (prod + 1) & 3;
    }
    // the WZ - 1 planes above the piece's last complete one, shared with the piece above
#pragma unroll
    for (int kk = 0; kk + 1 < WZ; ++kk) {
        red_pair(reinterpret_cast<P2*>(gcol + (size_t)pz * plane), acc[kk]);
        pz = pz + 1 == g.n ? 0 : pz + 1;
        acc[kk].x = (T)0; acc[kk].y = (T)0;
    }
    }
}

}  // namespace enuf
