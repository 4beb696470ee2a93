// Step a1 -- wrap positions (x = r/L; R10) and counting-sort the charged
// particles by bin (16 x 16 column in x, y and grid plane in z; TileGeom in enuf_common.cuh):
// histogram -> exclusive scan (one launch, or two for histograms of more chunks than SMs) -> scatter ->
// window rows of the sorted particles.  The cell index c and
// the fractional offset d0 = u - c are formed in fp64 in the order
//   x = r/L;  x -= floor(x);  u = n*x;  c = floor(u + 1/2)
// for both precisions (an fp32 u would lose the offset: ulp(256) ~ 1.5e-5 cells), so the
// binned record carries d0 to full precision of T.
#pragma once

#include "enuf_common.cuh"
#include "enuf_spread.cuh"   // WindowRows, write_window_row

namespace enuf {

struct CellOfParticle {
    int c[3];        // nearest grid point per dimension, wrapped into [0, n)
    double d0[3];    // u - (unwrapped c), in [-1/2, 1/2]
};

template <typename T>
__device__ __forceinline__ CellOfParticle locate(const T* __restrict__ r, int64_t j, const Edges& L, int n) {
    CellOfParticle o;
#pragma unroll
    for (int t = 0; t < 3; ++t) {
        double x = __ddiv_rn((double)r[3 * j + t], L.l[t]);
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

template <typename T>
__device__ __forceinline__ int bin_of(const CellOfParticle& p, const TileGeom& g) {
    int bz = p.c[2];
    if (g.trim) {       // the sign test is taken on the value the record stores (rounded to T)
        bz += ((T)p.d0[2] > (T)0 ? 1 : 0) - 1;
        bz += bz < 0 ? g.n : 0;
    }
    return bin_index(g, p.c[0] / kTile, p.c[1] / kTile, bz);
}

// Histogram of charged particles per bin; neutral particles get F = 0 here and are dropped.  The histogram atomic
// returns the particle's rank inside its bin: (bin, rank) is kept per particle, so that the scatter needs no atomic.
constexpr uint32_t kNoBin = 0xffffffffu;
template <typename T>
__global__ void __launch_bounds__(256)
bin_count_kernel(const T* __restrict__ r, const T* __restrict__ q, T* __restrict__ F, int64_t N,
                 Edges L, TileGeom g, uint32_t* __restrict__ count, uint32_t* __restrict__ scan_epoch,
                 uint2* __restrict__ binrank, unsigned zblocks, SpreadZero<T> zr) {
    pdl_prologue();
    // the first zblocks blocks clear the grid planes that two spreading pieces add into (enuf_spread.cuh); the first
    // kernel of the evaluation does it because the previous evaluation's gather is the grid's last reader
    if (blockIdx.x < zblocks) { spread_zero_block(zr, (int)blockIdx.x); return; }
    int64_t j = (int64_t)(blockIdx.x - zblocks) * blockDim.x + threadIdx.x;
    if (j >= N) return;
    if (j == 0) scan_epoch[0] += 1u;    // the epoch of this evaluation's scan: kept on the device so that a
                                        // replayed CUDA graph (ENUF_OPT_CUDA_GRAPH) advances it as well
    if (q[j] == (T)0) {
        F[3 * j] = (T)0; F[3 * j + 1] = (T)0; F[3 * j + 2] = (T)0;
        binrank[j] = make_uint2(kNoBin, 0u);
        return;
    }
    CellOfParticle p = locate(r, j, L, g.n);
    const uint32_t b = (uint32_t)bin_of<T>(p, g);
    binrank[j] = make_uint2(b, atomicAdd(&count[b], 1u));
}

// Exclusive scan of count[0..nbins) into offset[0..nbins] (and a copy in cursor[0..nbins),
// the scatter's running positions).  Two launches of kScanThreads threads per CTA, each
// CTA owning kScanChunk = 4 * kScanThreads consecutive bins:
//   bin_scan_totals: total[b] = sum of chunk b
//   bin_scan_apply : base = sum of total[< b] (few hundred values at most), then a CTA scan; it also
//                    clears count[] behind itself, so only the first evaluation needs a memset.
constexpr int kScanThreads = 256;
constexpr int kScanChunk = 4 * kScanThreads;

static __global__ void __launch_bounds__(kScanThreads)
bin_scan_totals_kernel(const uint32_t* __restrict__ count, int nbins, uint32_t* __restrict__ total) {
    pdl_prologue();
    __shared__ uint32_t ws[kScanThreads / 32];
    const int i0 = blockIdx.x * kScanChunk + threadIdx.x * 4;
    uint32_t v = 0;
#pragma unroll
    for (int e = 0; e < 4; ++e) if (i0 + e < nbins) v += count[i0 + e];
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
    if ((threadIdx.x & 31) == 0) ws[threadIdx.x >> 5] = v;
    __syncthreads();
    if (threadIdx.x == 0) {
        uint32_t s = 0;
#pragma unroll
        for (int w = 0; w < kScanThreads / 32; ++w) s += ws[w];
        total[blockIdx.x] = s;
    }
}

static __global__ void __launch_bounds__(kScanThreads)
bin_scan_apply_kernel(uint32_t* __restrict__ count, int nbins, const uint32_t* __restrict__ total,
                      uint32_t* __restrict__ offset, uint32_t* __restrict__ cursor) {
    pdl_prologue();
    __shared__ uint32_t ws[kScanThreads / 32];
    __shared__ uint32_t base_s;
    const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
    // base of this chunk
    uint32_t b = 0;
    for (int i = threadIdx.x; i < (int)blockIdx.x; i += kScanThreads) b += total[i];
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) b += __shfl_xor_sync(0xffffffffu, b, o);
    if (lane == 0) ws[wid] = b;
    __syncthreads();
    if (threadIdx.x == 0) {
        uint32_t s = 0;
#pragma unroll
        for (int w = 0; w < kScanThreads / 32; ++w) s += ws[w];
        base_s = s;
    }
    __syncthreads();
    const uint32_t base = base_s;
    __syncthreads();
    const int i0 = blockIdx.x * kScanChunk + threadIdx.x * 4;
    uint32_t c[4], sum = 0;
#pragma unroll
    for (int e = 0; e < 4; ++e) {
        c[e] = i0 + e < nbins ? count[i0 + e] : 0u;
        sum += c[e];
        if (i0 + e < nbins) count[i0 + e] = 0u;      // the histogram is left cleared for the next evaluation
    }
    uint32_t inc = sum;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
        uint32_t t = __shfl_up_sync(0xffffffffu, inc, o);
        if (lane >= o) inc += t;
    }
    if (lane == 31) ws[wid] = inc;
    __syncthreads();
    uint32_t wbase = 0;
#pragma unroll
    for (int w = 0; w < kScanThreads / 32; ++w) if (w < wid) wbase += ws[w];
    uint32_t run = base + wbase + inc - sum;
#pragma unroll
    for (int e = 0; e < 4; ++e) {
        if (i0 + e < nbins) { offset[i0 + e] = run; cursor[i0 + e] = run; }
        run += c[e];
    }
    if (i0 <= nbins - 1 && nbins - 1 < i0 + 4) offset[nbins] = run;   // thread owning the last bin
}

// Single-launch variant for histograms of at most kScanMaxResident chunks (every CTA is resident at once, so a
// CTA may wait for its predecessors): chunk b publishes (epoch << 32 | its total) in desc[b] and sums the
// totals of the chunks before it as they appear (decoupled look-back without the aggregate chain -- with <= 64
// chunks reading all predecessors is cheaper than chaining).  the epoch changes with every evaluation, so desc[] is
// never reset.
constexpr int kScanMaxResident = 128;
static __global__ void __launch_bounds__(kScanThreads)
bin_scan_single_kernel(uint32_t* __restrict__ count, int nbins, unsigned long long* __restrict__ desc,
                       const uint32_t* __restrict__ scan_epoch, uint32_t* __restrict__ offset,
                       uint32_t* __restrict__ cursor) {
    pdl_prologue();
    __shared__ uint32_t ws[kScanThreads / 32];
    __shared__ uint32_t base_s;
    const uint32_t epoch = scan_epoch[0];             // advanced by bin_count_kernel of this evaluation
    const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
    const int i0 = blockIdx.x * kScanChunk + threadIdx.x * 4;
    uint32_t c[4], sum = 0;
#pragma unroll
    for (int e = 0; e < 4; ++e) {
        c[e] = i0 + e < nbins ? count[i0 + e] : 0u;
        sum += c[e];
        if (i0 + e < nbins) count[i0 + e] = 0u;      // the histogram is left cleared for the next evaluation
    }
    // inclusive scan of the per-thread sums inside the CTA
    uint32_t inc = sum;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
        uint32_t t = __shfl_up_sync(0xffffffffu, inc, o);
        if (lane >= o) inc += t;
    }
    if (lane == 31) ws[wid] = inc;
    __syncthreads();
    uint32_t wbase = 0, ctot = 0;
#pragma unroll
    for (int w = 0; w < kScanThreads / 32; ++w) { if (w < wid) wbase += ws[w]; ctot += ws[w]; }
    if (threadIdx.x == 0) {
        __threadfence();
        atomicExch(&desc[blockIdx.x], ((unsigned long long)epoch << 32) | ctot);
    }
    // totals of the chunks before this one
    uint32_t part = 0;
    for (int i = threadIdx.x; i < (int)blockIdx.x; i += kScanThreads) {
        unsigned long long d;
        do { d = *reinterpret_cast<volatile unsigned long long*>(&desc[i]); } while ((uint32_t)(d >> 32) != epoch);
        part += (uint32_t)d;
    }
    __syncthreads();                                  // ws is reused
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) part += __shfl_xor_sync(0xffffffffu, part, o);
    if (lane == 0) ws[wid] = part;
    __syncthreads();
    if (threadIdx.x == 0) {
        uint32_t b = 0;
#pragma unroll
        for (int w = 0; w < kScanThreads / 32; ++w) b += ws[w];
        base_s = b;
    }
    __syncthreads();
    uint32_t run = base_s + wbase + inc - sum;
#pragma unroll
    for (int e = 0; e < 4; ++e) {
        if (i0 + e < nbins) { offset[i0 + e] = run; cursor[i0 + e] = run; }
        run += c[e];
    }
    if (i0 <= nbins - 1 && nbins - 1 < i0 + 4) offset[nbins] = run;   // thread owning the last bin
}

// Scatter into bin order: position = offset[bin] + rank, both from the count pass (no atomic here).  The order inside
// a bin is the arrival order at the histogram (any order is a valid sort; sums downstream differ only in rounding
// order, R22).  Bits 30 / 31 of the packed cell carry
// ks_x / ks_y = (d0 > 0) of the trimmed stencils (the spreading producer culls on the cell word alone).
template <typename T>
__global__ void __launch_bounds__(256)
bin_scatter_kernel(const T* __restrict__ r, const T* __restrict__ q, int64_t N, Edges L, TileGeom g,
                   const uint32_t* __restrict__ offset, const uint2* __restrict__ binrank, PSlot<T>* __restrict__ slots) {
    pdl_prologue();
    int64_t j = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (j >= N) return;
    const uint2 br = binrank[j];
    if (br.x == kNoBin) return;
    const T qj = q[j];
    CellOfParticle p = locate(r, j, L, g.n);
    const uint32_t pos = offset[br.x] + br.y;
    PSlot<T> o;
    o.rec.dx = (T)p.d0[0]; o.rec.dy = (T)p.d0[1]; o.rec.dz = (T)p.d0[2]; o.rec.q = qj;
    const uint32_t ksx = (g.trim && o.rec.dx > (T)0) ? 1u : 0u, ksy = (g.trim && o.rec.dy > (T)0) ? 1u : 0u;
    o.cell = pack_cell(p.c[0], p.c[1], p.c[2]) | (ksx << 30) | (ksy << 31);
    o.idx = (uint32_t)j;
    slots[pos] = o;
}

// The window rows of the sorted particles (enuf_spread.cuh, WindowRows): the 3 x (2m+1) window values of a
// particle are evaluated ONCE per evaluation here ("window values ... kept") and read by every
// spreading CTA whose halo holds the particle.  A CTA of three warps takes 32 consecutive sorted particles --
// warp d evaluates dimension d, one lane per particle -- and writes their rows, one contiguous block, with
// coalesced 16-byte stores through a shared-memory transpose.
constexpr int kRowsThreads = 96;
template <typename T, int M_, bool kTrim>
__global__ void __launch_bounds__(kRowsThreads)
window_rows_kernel(const PSlot<T>* __restrict__ slots, const uint32_t* __restrict__ offset, int nbins, WindowParams wp,
                   const __grid_constant__ PolyArg<M_> pa, T* __restrict__ rows) {
    pdl_prologue();
    using R = WindowRows<M_, kTrim>;
    using V4 = typename Vec4<T>::type;
    constexpr int SP = R::RP + 4;                                  // 44 / 52 elements: conflict-free 16-byte accesses
    __shared__ __align__(16) T tile[32 * SP];
    const int lane = threadIdx.x & 31, dim = threadIdx.x >> 5;
    const uint32_t n_charged = offset[nbins];
    const uint32_t base = (uint32_t)blockIdx.x * 32u;
    if (base >= n_charged) return;
    const uint32_t nv = min(32u, n_charged - base);
    if ((uint32_t)lane < nv) {
        const PSlot<T> sl = slots[base + lane];
        const int ksx = (int)((sl.cell >> 30) & 1u);
        // parity of the first x stencil point (grid index c_x - m + ks_x; n is even, so wrapping keeps it)
        const int parx = ((int)(sl.cell & 1023u) + M_ + ksx) & 1;
        const T d0 = dim == 0 ? sl.rec.dx : (dim == 1 ? sl.rec.dy : sl.rec.dz);
        write_window_row<T, M_, kTrim>(wp, pa, dim, d0, sl.rec.q, parx, tile + lane * SP);
    }
    __syncthreads();
    T* out = rows + (size_t)base * R::RP;
    constexpr int CH = R::RP / 4;                                  // 16-byte (fp32) / 32-byte (fp64) chunks per particle
    for (int c = threadIdx.x; c < (int)nv * CH; c += kRowsThreads) {
        const int pp = c / CH, cc = c - pp * CH;
        reinterpret_cast<V4*>(out)[c] = reinterpret_cast<const V4*>(tile + pp * SP)[cc];
    }
}

// Scatter and window rows in one pass over the particles in CALLER order, for systems of at most kBinFusedMaxN particles
// (launch_bin, enuf_launch.cuh; larger ones run the two kernels above): a CTA of three warps takes 32 consecutive particles, warp d locates dimension d of
// particle `lane` (cell index and offset, fp64 as in locate()), the three meet in shared memory, warp 0 writes the
// sorted-array slot at offset[bin] + rank and warp d evaluates the particle's window row of dimension d; the rows leave
// as 16-byte stores, RP / 4 consecutive threads per particle (one particle's rows are contiguous, the particles of a
// CTA land wherever their bins are).  Against bin_scatter + window_rows this saves the second pass over the slots
// and one launch; the scattered 160-byte row blocks cost more than that once N reaches ~1e6.
constexpr int64_t kBinFusedMaxN = 262144;
template <typename T, int M_, bool kTrim>
__global__ void __launch_bounds__(kRowsThreads)
bin_place_kernel(const T* __restrict__ r, const T* __restrict__ q, int64_t N, Edges L, TileGeom g,
                 const uint32_t* __restrict__ offset, const uint2* __restrict__ binrank, PSlot<T>* __restrict__ slots,
                 WindowParams wp, const __grid_constant__ PolyArg<M_> pa, T* __restrict__ rows) {
    pdl_prologue();
    using R = WindowRows<M_, kTrim>;
    using V4 = typename Vec4<T>::type;
    constexpr int SP = R::RP + 4;                                  // 44 / 52 elements: conflict-free 16-byte accesses
    __shared__ __align__(16) T tile[32 * SP];
    __shared__ T d0_s[3][32];
    __shared__ int c_s[3][32];
    __shared__ uint32_t pos_s[32];
    const int lane = threadIdx.x & 31, dim = threadIdx.x >> 5;
    const int64_t j = (int64_t)blockIdx.x * 32 + lane;
    uint2 br = make_uint2(kNoBin, 0u);
    if (j < N) br = binrank[j];
    const bool live = br.x != kNoBin;
    T d0 = (T)0, qj = (T)0;
    int ci = 0;
    if (live) {
        // one dimension of locate(): x = r/L; x -= floor(x); u = n x; c = floor(u + 1/2); d0 = u - c
        double x = __ddiv_rn((double)r[3 * j + dim], L.l[dim]);
        x -= floor(x);
        if (x >= 1.0) x = 0.0;
        const double u = __dmul_rn((double)g.n, x);
        const double c = floor(__dadd_rn(u, 0.5));
        d0 = (T)(u - c);
        ci = (int)c;
        ci = ci >= g.n ? ci - g.n : ci;
        qj = q[j];
        d0_s[dim][lane] = d0;
        c_s[dim][lane] = ci;
        if (dim == 0) pos_s[lane] = offset[br.x] + br.y;
    } else if (dim == 0) {
        pos_s[lane] = 0xffffffffu;
    }
    __syncthreads();
    if (live) {
        const int ksx = (kTrim && d0_s[0][lane] > (T)0) ? 1 : 0;
        if (dim == 0) {
            PSlot<T> o;
            o.rec.dx = d0_s[0][lane]; o.rec.dy = d0_s[1][lane]; o.rec.dz = d0_s[2][lane]; o.rec.q = qj;
            const uint32_t ksy = (kTrim && o.rec.dy > (T)0) ? 1u : 0u;
            o.cell = pack_cell(c_s[0][lane], c_s[1][lane], c_s[2][lane]) | ((uint32_t)ksx << 30) | (ksy << 31);
            o.idx = (uint32_t)j;
            slots[pos_s[lane]] = o;
        }
        // parity of the first x stencil point (grid index c_x - m + ks_x; n is even, so wrapping keeps it)
        const int parx = (c_s[0][lane] + M_ + ksx) & 1;
        write_window_row<T, M_, kTrim>(wp, pa, dim, d0, qj, parx, tile + lane * SP);
    }
    __syncthreads();
    constexpr int CH = R::RP / 4;                                  // 16-byte (fp32) / 32-byte (fp64) chunks per particle
    for (int c = threadIdx.x; c < 32 * CH; c += kRowsThreads) {
        const int pp = c / CH, cc = c - pp * CH;
        const uint32_t pos = pos_s[pp];
        if (pos != 0xffffffffu)
            reinterpret_cast<V4*>(rows + (size_t)pos * R::RP)[cc] = reinterpret_cast<const V4*>(tile + pp * SP)[cc];
    }
}

}  // namespace enuf
