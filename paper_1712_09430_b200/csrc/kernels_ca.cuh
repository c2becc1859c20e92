// K1 cluster sort + row grid, K2 neighbours finder, K3/K4 neighbours cleaner + start-hit finder.
// Phase I step 1, "seeding ... heuristics in a cellular automaton", one GPU thread per hit
// (PAPER.md:33,66); readings S1..S4 of DESIGN.md.  Compiled with -fmad=false: every decision value is the
// IEEE fp32 result of the written expression (R-12).
#pragma once
#include "device_types.cuh"

namespace tpc {

// Bin index of coordinate v: monotone non-decreasing in v, total (NaN -> 0), used for hits AND queries.
__device__ __forceinline__ int bin_of(float v, float v0, float inv, int n) {
    float f = (v - v0) * inv;
    f = fminf(fmaxf(f, 0.0f), (float)(n - 1));
    return (int)f;
}

// ------------------------------------------------------------------------------------------ K1
// One block per (sector,row): bounding box -> grid -> histogram in shared memory -> scan -> scatter.
// Input: SoA y[], z[] as loaded (coalesced reads).  Output: sorted float2 (y,z), orig[], binStart[], grid.
#ifndef TPC_ZF
#define TPC_ZF 2.1f   /* measured on config 3 (K5 us), 3 bins per hit: 1.5 -> 847, 1.8 -> 590, 2.2 -> 497, 2.6 -> 509; 2 bins per hit:
                         1.9 -> 368, 2.0 -> 361, 2.1 -> 362, 2.2 -> 363, 2.3 -> 366, 2.4 -> 368, 2.7 -> 372; the steep side is the low one */
#endif
#ifndef TPC_K1T
#define TPC_K1T 160   /* threads per (sector,row) block; K1 us on config 3: 64 -> 53.5, 96 -> 49.6, 128 -> 45.6, 160 -> 44.0, 192 -> 47.6, 256 -> 51.7 */
#endif
constexpr int kK1Threads = TPC_K1T;
constexpr int kK1Stage = 512;     // 8 KB of static shared memory beside the <= 32 KB dynamic histogram (48 KB limit)

__global__ void __launch_bounds__(kK1Threads) k1_sort_grid(DevPtrs d) {
    const int rowId = blockIdx.x;
    const int tid = threadIdx.x;
    if (rowId == 0 && tid < kNCounters) d.counters[tid] = 0u;
    if (rowId == 0) for (int i = tid; i <= kMaxRows; i += kK1Threads) d.rowHist[i] = 0u;
    const RowMeta M = d.meta[rowId];
    RowGrid R = d.grid[rowId];
    const int n = M.n;
    if (n == 0) {   // empty row: the host's default 1x1 grid stays; give it an empty bucket
        if (tid == 0) {
            const float qn = __int_as_float(0x7fc00000);
            float4* q = reinterpret_cast<float4*>(d.buckets + R.binOff);
            q[0] = make_float4(0.f, 0.f, qn, qn);
            q[1] = make_float4(qn, qn, qn, qn);
            d.binStart[R.binOff] = 0u; d.binStart[R.binOff + 1] = 0u;
        }
        return;
    }
    extern __shared__ uint32_t sh[];            // [maxBins + 1] histogram / cursors
    __shared__ float redA[4][kK1Threads / 32];
    __shared__ float redZ[kK1Threads / 32];
    // rows of up to kK1Stage hits keep their input and their sorted hits in shared memory, so that the three passes
    // over the input and the bucket pass do not go back to global memory (each pass is one more dependent memory
    // round trip in a block's life); larger rows re-read global memory
    __shared__ float2 sIn[kK1Stage];
    __shared__ float2 sSorted[kK1Stage];
    const bool staged = n <= kK1Stage;
    __shared__ uint32_t warpSum[kK1Threads / 32];
    __shared__ int sNY, sNZ;
    __shared__ float sY0, sZ0, sInvY, sInvZ;
    const float* __restrict__ y = d.inY + M.inOff;
    const float* __restrict__ z = d.inZ + M.inOff;

    // 1. bounding box
    float ymin = 3.0e38f, ymax = -3.0e38f, zmin = 3.0e38f, zmax = -3.0e38f;
    float zsum = 0.0f;
    for (int i = tid; i < n; i += kK1Threads) {
        const float a = y[i], b = z[i];
        ymin = fminf(ymin, a); ymax = fmaxf(ymax, a);
        zmin = fminf(zmin, b); zmax = fmaxf(zmax, b);
        zsum += b;
        if (staged) sIn[i] = make_float2(a, b);
    }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) {
        zsum += __shfl_xor_sync(0xffffffffu, zsum, o);
        ymin = fminf(ymin, __shfl_xor_sync(0xffffffffu, ymin, o));
        ymax = fmaxf(ymax, __shfl_xor_sync(0xffffffffu, ymax, o));
        zmin = fminf(zmin, __shfl_xor_sync(0xffffffffu, zmin, o));
        zmax = fmaxf(zmax, __shfl_xor_sync(0xffffffffu, zmax, o));
    }
    if ((tid & 31) == 0) { redA[0][tid >> 5] = ymin; redA[1][tid >> 5] = ymax; redA[2][tid >> 5] = zmin; redA[3][tid >> 5] = zmax; redZ[tid >> 5] = zsum; }
    __syncthreads();
    if (tid == 0) {
        for (int w = 1; w < kK1Threads / 32; w++) {
            ymin = fminf(ymin, redA[0][w]); ymax = fmaxf(ymax, redA[1][w]);
            zmin = fminf(zmin, redA[2][w]); zmax = fmaxf(zmax, redA[3][w]);
            zsum += redZ[w];
        }
        // non-finite input must not blow the grid up
        ymin = fminf(fmaxf(ymin, -1.0e4f), 1.0e4f); ymax = fminf(fmaxf(ymax, -1.0e4f), 1.0e4f);
        zmin = fminf(fmaxf(zmin, -1.0e4f), 1.0e4f); zmax = fminf(fmaxf(zmax, -1.0e4f), 1.0e4f);
        // The grid need not cover every hit: bin_of clamps, so hits (and queries) beyond the grid's range fall into
        // its edge bins.  In z the occupancy is lopsided - tracks fill |z| < ~x, noise the whole drift length - so
        // the z-range is cut to TPC_ZF x the distance from the denser end to the mean: the bins get finer where the
        // tracks are, for the same number of bins (a uniform or symmetric distribution keeps its full range).
        const float zmean = zsum / (float)n;
        if (zmean > zmin && zmean < zmax) {
            const float a = zmean - zmin, b = zmax - zmean;
            if (a < b) zmax = fminf(zmax, zmin + TPC_ZF * a);
            else zmin = fmaxf(zmin, zmax - TPC_ZF * b);
        }
        const float spanY = fmaxf(ymax - ymin, 1.0e-2f), spanZ = fmaxf(zmax - zmin, 1.0e-2f);
        // kBinsPerHit bins per hit, bins twice as long in z as in y (a query costs per z-bin-row), >= 0.5 cm
        const int target = max(1, M.maxBins);
        float ey = sqrtf(spanY * spanZ / (2.0f * (float)target));
        ey = fmaxf(ey, 0.5f);
        int nY = max(1, min(target, (int)(spanY / ey)));
        int nZ = max(1, min(target / nY, (int)(spanZ / (2.0f * ey))));
        sNY = nY; sNZ = nZ; sY0 = ymin; sZ0 = zmin;
        sInvY = (float)nY / spanY; sInvZ = (float)nZ / spanZ;
        R.nY = nY; R.nZ = nZ; R.y0 = ymin; R.z0 = zmin; R.invY = sInvY; R.invZ = sInvZ;
        d.grid[rowId] = R;
    }
    __syncthreads();
    const int nY = sNY, nZ = sNZ, nBins = nY * nZ;
    const float y0 = sY0, z0 = sZ0, invY = sInvY, invZ = sInvZ;

    // 2. histogram
    for (int b = tid; b <= nBins; b += kK1Threads) sh[b] = 0u;
    __syncthreads();
    for (int i = tid; i < n; i += kK1Threads) {
        const float2 v = staged ? sIn[i] : make_float2(y[i], z[i]);
        const int b = bin_of(v.y, z0, invZ, nZ) * nY + bin_of(v.x, y0, invY, nY);
        atomicAdd(&sh[b], 1u);
    }
    __syncthreads();

    // 3. exclusive scan of sh[0..nBins] (chunk per thread, warp shuffles across chunks)
    const int chunk = (nBins + 1 + kK1Threads - 1) / kK1Threads;
    const int b0 = min(tid * chunk, nBins + 1), b1 = min(b0 + chunk, nBins + 1);
    uint32_t local = 0;
    for (int b = b0; b < b1; b++) local += sh[b];
    uint32_t incl = local;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
        const uint32_t v = __shfl_up_sync(0xffffffffu, incl, o);
        if ((tid & 31) >= o) incl += v;
    }
    if ((tid & 31) == 31) warpSum[tid >> 5] = incl;
    __syncthreads();
    uint32_t base = incl - local;
    for (int w = 0; w < (tid >> 5); w++) base += warpSum[w];
    uint32_t* __restrict__ bs = d.binStart + R.binOff;
    for (int b = b0; b < b1; b++) {
        const uint32_t c = sh[b];
        sh[b] = base;          // becomes the scatter cursor
        bs[b] = base;
        base += c;
    }
    __syncthreads();

    // 4. scatter (order inside a bin is arbitrary: no result depends on it, tie-breaks use orig[])
    float2* __restrict__ hs = d.hits + R.hitOff;
    uint32_t* __restrict__ og = d.orig + R.hitOff;
    uint32_t* __restrict__ wt = d.weight + R.hitOff;
    for (int i = tid; i < n; i += kK1Threads) {
        const float2 v = staged ? sIn[i] : make_float2(y[i], z[i]);
        const float a = v.x, c = v.y;
        const int b = bin_of(c, z0, invZ, nZ) * nY + bin_of(a, y0, invY, nY);
        const uint32_t pos = atomicAdd(&sh[b], 1u);
        hs[pos] = make_float2(a, c);
        if (staged) sSorted[pos] = make_float2(a, c);
        og[pos] = M.gidBase + (uint32_t)i;
        wt[i] = 0u;
    }
    __syncthreads();

    // 5. buckets: after the scatter sh[b] is the END of bin b, so bin b starts at sh[b-1]
    Bucket* __restrict__ bk = d.buckets + R.binOff;
    const float qnan = __int_as_float(0x7fc00000);
    for (int b = tid; b < nBins; b += kK1Threads) {
        const uint32_t s0 = b ? sh[b - 1] : 0u, cnt = sh[b] - s0;
        float2 h0 = make_float2(qnan, qnan), h1 = h0, h2 = h0;   // NaN never passes a window test
        if (cnt > 0) h0 = staged ? sSorted[s0] : hs[s0];
        if (cnt > 1) h1 = staged ? sSorted[s0 + 1] : hs[s0 + 1];
        if (cnt > 2) h2 = staged ? sSorted[s0 + 2] : hs[s0 + 2];
        float4* q = reinterpret_cast<float4*>(bk + b);
        q[0] = make_float4(__uint_as_float(s0), __uint_as_float(cnt), h0.x, h0.y);
        q[1] = make_float4(h1.x, h1.y, h2.x, h2.y);
    }
}

// Enumerate every hit of row R whose bin overlaps [yc-wy, yc+wy] x [zc-wz, zc+wz] (a superset of the window).
template <class F>
__device__ __forceinline__ void for_window(const RowGrid& R, const float2* __restrict__ hits,
                                           const uint32_t* __restrict__ binStart, float yc, float zc, float wy,
                                           float wz, F&& f) {
    const int by0 = bin_of(yc - wy - kGridMargin, R.y0, R.invY, R.nY);
    const int by1 = bin_of(yc + wy + kGridMargin, R.y0, R.invY, R.nY);
    const int bz0 = bin_of(zc - wz - kGridMargin, R.z0, R.invZ, R.nZ);
    const int bz1 = bin_of(zc + wz + kGridMargin, R.z0, R.invZ, R.nZ);
    const uint32_t* __restrict__ bs = binStart + R.binOff;
    const float2* __restrict__ hs = hits + R.hitOff;
    for (int bz = bz0; bz <= bz1; bz++) {
        const int k0 = (int)bs[bz * R.nY + by0], k1 = (int)bs[bz * R.nY + by1 + 1];
        for (int k = k0; k < k1; k++) f(k, hs[k]);
    }
}

// The same enumeration in two steps, for K2: win_ranges() requests the bin-table entries of up to three z-rows of
// bins at once (six independent loads; both adjacent rows' windows are requested before either is scanned), scan_ranges()
// then walks the hit ranges.  Windows taller than three bin rows take the generic loop.
struct WinRanges {
    int k0[3], k1[3];
    int by0, by1, bz0, bz1;
};
__device__ __forceinline__ WinRanges win_ranges(const RowGrid& R, const uint32_t* __restrict__ binStart, float yc,
                                                float zc, float wy, float wz) {
    WinRanges w;
    w.by0 = bin_of(yc - wy - kGridMargin, R.y0, R.invY, R.nY);
    w.by1 = bin_of(yc + wy + kGridMargin, R.y0, R.invY, R.nY);
    w.bz0 = bin_of(zc - wz - kGridMargin, R.z0, R.invZ, R.nZ);
    w.bz1 = bin_of(zc + wz + kGridMargin, R.z0, R.invZ, R.nZ);
    const uint32_t* __restrict__ bs = binStart + R.binOff;
#pragma unroll
    for (int j = 0; j < 3; j++) {
        const int bz = min(w.bz0 + j, w.bz1);           // rows beyond the window repeat the last one (valid address)
        const bool in = w.bz0 + j <= w.bz1;
        const int a = (int)bs[bz * R.nY + w.by0], b = (int)bs[bz * R.nY + w.by1 + 1];
        w.k0[j] = in ? a : 0;
        w.k1[j] = in ? b : 0;
    }
    return w;
}
template <class F>
__device__ __forceinline__ void scan_ranges(const WinRanges& w, const RowGrid& R, const float2* __restrict__ hits,
                                            const uint32_t* __restrict__ binStart, F&& f) {
    const float2* __restrict__ hs = hits + R.hitOff;
    if (w.bz1 - w.bz0 <= 2) {
        // one loop over the three ranges laid end to end: the warp runs max over lanes of the TOTAL length, not the
        // sum over ranges of the per-range maxima
        const int l0 = w.k1[0] - w.k0[0], l1 = l0 + (w.k1[1] - w.k0[1]), l2 = l1 + (w.k1[2] - w.k0[2]);
        const int o1 = w.k0[1] - l0, o2 = w.k0[2] - l1;
        auto at = [&](int t) { return t < l0 ? w.k0[0] + t : t < l1 ? o1 + t : o2 + t; };
        if (l2 > 0) {
            int k = at(0);
            float2 c = hs[k];
            for (int t = 0; t < l2; t++) {
                const int kn = at(min(t + 1, l2 - 1));      // next candidate requested before this one is examined
                const float2 cn = hs[kn];
                f(k, c);
                k = kn; c = cn;
            }
        }
    } else {
        const uint32_t* __restrict__ bs = binStart + R.binOff;
        for (int bz = w.bz0; bz <= w.bz1; bz++) {
            const int k0 = (int)bs[bz * R.nY + w.by0], k1 = (int)bs[bz * R.nY + w.by1 + 1];
            for (int k = k0; k < k1; k++) f(k, hs[k]);
        }
    }
}

// ------------------------------------------------------------------------------------------ K2
// Neighbours finder (S2): for each hit the best (up,down) pair in rows r+1/r-1 by 3-point collinearity; one thread
// per hit.
//
// A block takes a CHUNK of up to kK2Chunk consecutive sorted hits of one (sector,row) (a row of a time frame holds
// ~5,500 hits: one block per row left most SMs waiting for the longest rows, 15.3 -> 10.0 ms for K2 there).  K1 sorted
// the hits by bin, z-major, so a chunk covers a band in z, and everything its hits can reach in an adjacent row - the
// rows of bins that overlap [zmin - window, zmax + window] - is ONE contiguous piece of that row's sorted hits and of
// its bin table.
// kStage (tpc_set_neighbour_staging, OFF by default): those two pieces per adjacent row are staged in shared memory
// first, the hits with a 1-D bulk copy (cp.async.bulk + mbarrier: the TMA engine), the bin table with coalesced
// loads; every candidate scan then reads shared memory.  A piece that does not fit (kK2StageHits / kK2StageBins)
// makes the block read global memory like the unstaged instantiation (same code, other pointers).  Measured, it
// loses: 120 vs 90 us on a central event, 11.4 vs 10.0 ms on a time frame - a block's work is a few microseconds
// (2-3 hits per thread), and the z-band pass, the barrier and the wait for the copies stand in front of all of it,
// while the unstaged scans already hit L1 for 77 % of their sectors (profiles/r02_k2_staging.md has both columns).
#ifndef TPC_K2T
#define TPC_K2T 128
#endif
constexpr int kK2Threads = TPC_K2T;
#ifndef TPC_K2CAP
#define TPC_K2CAP 8
#endif
constexpr int kK2Cap = TPC_K2CAP;   // down-candidates cached per thread (registers); beyond that a grid query per up-candidate
#ifndef TPC_K2CAPD
#define TPC_K2CAPD 12
#endif
constexpr int kK2CapDense = TPC_K2CAPD;   // ... in the instantiation for dense rows (time frames: ~20x the candidates per window).
// Measured (central event K2 us / time frame K2 ms), grid query on: cap 8: 83.7 / 7.2, 10: 88.6 / 6.6, 12: 95.5 / 6.4,
// 16: 104.8 / 6.5; with the whole-window rescan it replaced, cap 8: 89.5 / 8.9
#ifndef TPC_K2B
#define TPC_K2B 8
#endif
#ifndef TPC_K2CHUNK
#define TPC_K2CHUNK 256   /* 128 / 256 / 512 / 1024: K2 90.8 / 89.5 / 91.7 / 91.5 us (central event), 10.2 / 9.9 / 10.0 / 10.6 ms (time frame) */
#endif
constexpr int kK2Chunk = TPC_K2CHUNK;
constexpr int kK2StageHits = 1024;      // staged hits of each adjacent row (8 KB)
constexpr int kK2StageBins = 1280;      // staged bin-table entries of each adjacent row (5 KB)

// One adjacent row as the scans see it: hs[k - kBase] is sorted hit k, bs[b - bBase] is bin-table entry b.
struct K2Row {
    const float2* hs;
    const uint32_t* bs;
    int kBase, bBase;
};
__device__ __forceinline__ WinRanges k2_win_ranges(const RowGrid& R, const K2Row& V, float yc, float zc, float wy, float wz) {
    WinRanges w;
    w.by0 = bin_of(yc - wy - kGridMargin, R.y0, R.invY, R.nY);
    w.by1 = bin_of(yc + wy + kGridMargin, R.y0, R.invY, R.nY);
    w.bz0 = bin_of(zc - wz - kGridMargin, R.z0, R.invZ, R.nZ);
    w.bz1 = bin_of(zc + wz + kGridMargin, R.z0, R.invZ, R.nZ);
    const uint32_t* __restrict__ bs = V.bs - V.bBase;
#pragma unroll
    for (int j = 0; j < 3; j++) {
        const int bz = min(w.bz0 + j, w.bz1);           // rows beyond the window repeat the last one (valid address)
        const bool in = w.bz0 + j <= w.bz1;
        const int a = (int)bs[bz * R.nY + w.by0], b = (int)bs[bz * R.nY + w.by1 + 1];
        w.k0[j] = in ? a : 0;
        w.k1[j] = in ? b : 0;
    }
    return w;
}
template <class F>
__device__ __forceinline__ void k2_scan(const WinRanges& w, const RowGrid& R, const K2Row& V, F&& f) {
    const float2* __restrict__ hs = V.hs - V.kBase;
    if (w.bz1 - w.bz0 <= 2) {
        // one loop over the three ranges laid end to end: the warp runs max over lanes of the TOTAL length, not the
        // sum over ranges of the per-range maxima
        const int l0 = w.k1[0] - w.k0[0], l1 = l0 + (w.k1[1] - w.k0[1]), l2 = l1 + (w.k1[2] - w.k0[2]);
        const int o1 = w.k0[1] - l0, o2 = w.k0[2] - l1;
        auto at = [&](int t) { return t < l0 ? w.k0[0] + t : t < l1 ? o1 + t : o2 + t; };
        if (l2 > 0) {
            int k = at(0);
            float2 c = hs[k];
            for (int t = 0; t < l2; t++) {
                const int kn = at(min(t + 1, l2 - 1));      // next candidate requested before this one is examined
                const float2 cn = hs[kn];
                f(k, c);
                k = kn; c = cn;
            }
        }
    } else {
        const uint32_t* __restrict__ bs = V.bs - V.bBase;
        for (int bz = w.bz0; bz <= w.bz1; bz++) {
            const int k0 = (int)bs[bz * R.nY + w.by0], k1 = (int)bs[bz * R.nY + w.by1 + 1];
            for (int k = k0; k < k1; k++) f(k, hs[k]);
        }
    }
}
template <class F>
__device__ __forceinline__ void k2_for_window(const RowGrid& R, const K2Row& V, float yc, float zc, float wy, float wz, F&& f) {
    const int by0 = bin_of(yc - wy - kGridMargin, R.y0, R.invY, R.nY);
    const int by1 = bin_of(yc + wy + kGridMargin, R.y0, R.invY, R.nY);
    const int bz0 = bin_of(zc - wz - kGridMargin, R.z0, R.invZ, R.nZ);
    const int bz1 = bin_of(zc + wz + kGridMargin, R.z0, R.invZ, R.nZ);
    const uint32_t* __restrict__ bs = V.bs - V.bBase;
    const float2* __restrict__ hs = V.hs - V.kBase;
    for (int bz = bz0; bz <= bz1; bz++) {
        const int k0 = (int)bs[bz * R.nY + by0], k1 = (int)bs[bz * R.nY + by1 + 1];
        for (int k = k0; k < k1; k++) f(k, hs[k]);
    }
}

// the same for a box given by its bounds (nothing if a bound pair is crossed)
template <class F>
__device__ __forceinline__ void k2_for_box(const RowGrid& R, const K2Row& V, float ylo, float yhi, float zlo, float zhi, F&& f) {
    const int by0 = bin_of(ylo - kGridMargin, R.y0, R.invY, R.nY);
    const int by1 = bin_of(yhi + kGridMargin, R.y0, R.invY, R.nY);
    const int bz0 = bin_of(zlo - kGridMargin, R.z0, R.invZ, R.nZ);
    const int bz1 = bin_of(zhi + kGridMargin, R.z0, R.invZ, R.nZ);
    if (by0 > by1) return;
    const uint32_t* __restrict__ bs = V.bs - V.bBase;
    const float2* __restrict__ hs = V.hs - V.kBase;
    for (int bz = bz0; bz <= bz1; bz++) {
        const int k0 = (int)bs[bz * R.nY + by0], k1 = (int)bs[bz * R.nY + by1 + 1];
        for (int k = k0; k < k1; k++) f(k, hs[k]);
    }
}

__device__ __forceinline__ uint32_t smem_u32(const void* p) { return (uint32_t)__cvta_generic_to_shared(p); }

template <bool kStage, int kCap>
__global__ void __launch_bounds__(kK2Threads, TPC_K2B) k2_neighbours(DevPtrs d, DevParams dp) {
    __shared__ __align__(16) float2 sHitsU[kStage ? kK2StageHits : 1], sHitsD[kStage ? kK2StageHits : 1];
    __shared__ uint32_t sBinsU[kStage ? kK2StageBins : 1], sBinsD[kStage ? kK2StageBins : 1];
    __shared__ __align__(8) unsigned long long sBar;
    __shared__ float sRedLo[kK2Threads / 32], sRedHi[kK2Threads / 32];
    grid_dep_wait();
    const int rowId = blockIdx.x;
    const int r = rowId % dp.nRows;
    const int n = d.meta[rowId].n;
    const int i0 = blockIdx.y * kK2Chunk;
    if (i0 >= n) return;
    const int i1 = min(n, i0 + kK2Chunk);
    const RowGrid R = d.grid[rowId];
    int32_t* __restrict__ up = d.linkUp + R.hitOff;
    int32_t* __restrict__ dn = d.linkDn + R.hitOff;
    bool active = (r >= 1 && r <= dp.nRows - 2);
    RowGrid Ru = R, Rd = R;
    if (active) {
        Ru = d.grid[rowId + 1]; Rd = d.grid[rowId - 1];
        active = d.meta[rowId + 1].n > 0 && d.meta[rowId - 1].n > 0;
    }
    if (!active) {
        for (int i = i0 + threadIdx.x; i < i1; i += kK2Threads) { up[i] = -1; dn[i] = -1; }
        return;
    }
    const float xr = d.rowX[r];
    const float dxu = d.rowX[r + 1] - xr;
    const float dxd = d.rowX[r - 1] - xr;
    const float wu = -dxd / (dxu - dxd), wd = dxu / (dxu - dxd);
    const float wyU = dp.P.nf_ty * dxu + dp.P.nf_c, wzU = dp.P.nf_tz * dxu + dp.P.nf_c;
    const float wyD = dp.P.nf_ty * (-dxd) + dp.P.nf_c, wzD = dp.P.nf_tz * (-dxd) + dp.P.nf_c;
    const float rwd = 1.0f / wd;
    const float boxR = sqrtf(dp.P.nf_d2max) * rwd * 1.001f + 2.0e-3f;      // (see the rescan below)
    const uint32_t* __restrict__ origU = d.orig + Ru.hitOff;
    const uint32_t* __restrict__ origD = d.orig + Rd.hitOff;
    K2Row VU{d.hits + Ru.hitOff, d.binStart + Ru.binOff, 0, 0}, VD{d.hits + Rd.hitOff, d.binStart + Rd.binOff, 0, 0};

    if constexpr (kStage) {
        // z band of the chunk (its hits are read again below: L1)
        float zlo = 3.0e38f, zhi = -3.0e38f;
        for (int i = i0 + threadIdx.x; i < i1; i += kK2Threads) {
            const float z = d.hits[R.hitOff + i].y;
            zlo = fminf(zlo, z); zhi = fmaxf(zhi, z);
        }
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) {
            zlo = fminf(zlo, __shfl_xor_sync(0xffffffffu, zlo, o));
            zhi = fmaxf(zhi, __shfl_xor_sync(0xffffffffu, zhi, o));
        }
        if ((threadIdx.x & 31) == 0) { sRedLo[threadIdx.x >> 5] = zlo; sRedHi[threadIdx.x >> 5] = zhi; }
        if (threadIdx.x == 0) {
            asm volatile("mbarrier.init.shared::cta.b64 [%0], 1;" ::"r"(smem_u32(&sBar)));
            asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
        }
        __syncthreads();
#pragma unroll
        for (int w = 0; w < kK2Threads / 32; w++) { zlo = fminf(zlo, sRedLo[w]); zhi = fmaxf(zhi, sRedHi[w]); }
        // the pieces: rows of bins [bLo, bHi] of each neighbour, hits [k0, k1)
        const int uLo = bin_of(zlo - wzU - kGridMargin, Ru.z0, Ru.invZ, Ru.nZ), uHi = bin_of(zhi + wzU + kGridMargin, Ru.z0, Ru.invZ, Ru.nZ);
        const int dLo = bin_of(zlo - wzD - kGridMargin, Rd.z0, Rd.invZ, Rd.nZ), dHi = bin_of(zhi + wzD + kGridMargin, Rd.z0, Rd.invZ, Rd.nZ);
        const int ubBase = uLo * Ru.nY, ubCnt = (uHi - uLo + 1) * Ru.nY + 1;
        const int dbBase = dLo * Rd.nY, dbCnt = (dHi - dLo + 1) * Rd.nY + 1;
        const int uk0 = (int)VU.bs[ubBase] & ~1, uk1 = (int)VU.bs[ubBase + ubCnt - 1];      // (16-byte aligned start)
        const int dk0 = (int)VD.bs[dbBase] & ~1, dk1 = (int)VD.bs[dbBase + dbCnt - 1];
        const int uLen = (uk1 - uk0 + 1) & ~1, dLen = (dk1 - dk0 + 1) & ~1;                  // (whole 16-byte units)
        const bool fits = ubCnt <= kK2StageBins && dbCnt <= kK2StageBins && uLen <= kK2StageHits && dLen <= kK2StageHits;
        if (fits) {
            if (threadIdx.x == 0) {
                const uint32_t bytes = (uint32_t)(uLen + dLen) * (uint32_t)sizeof(float2);
                asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(&sBar)), "r"(bytes) : "memory");
                if (uLen > 0)
                    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];"
                                 ::"r"(smem_u32(sHitsU)), "l"(VU.hs + uk0), "r"((uint32_t)uLen * (uint32_t)sizeof(float2)), "r"(smem_u32(&sBar)) : "memory");
                if (dLen > 0)
                    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];"
                                 ::"r"(smem_u32(sHitsD)), "l"(VD.hs + dk0), "r"((uint32_t)dLen * (uint32_t)sizeof(float2)), "r"(smem_u32(&sBar)) : "memory");
            }
            for (int b = threadIdx.x; b < ubCnt; b += kK2Threads) sBinsU[b] = VU.bs[ubBase + b];
            for (int b = threadIdx.x; b < dbCnt; b += kK2Threads) sBinsD[b] = VD.bs[dbBase + b];
            {   // wait for the bulk copies (phase 0 of the barrier)
                uint32_t done = 0;
                while (!done)
                    asm volatile("{\n .reg .pred p;\n mbarrier.try_wait.parity.shared::cta.b64 p, [%1], 0;\n selp.u32 %0, 1, 0, p;\n}"
                                 : "=r"(done) : "r"(smem_u32(&sBar)) : "memory");
            }
            __syncthreads();
            VU = K2Row{sHitsU, sBinsU, uk0, ubBase};
            VD = K2Row{sHitsD, sBinsD, dk0, dbBase};
        }
    }

    for (int i = i0 + threadIdx.x; i < i1; i += kK2Threads) {
        const float2 h = d.hits[R.hitOff + i];
        float cy[kCap], cz[kCap];
        int ck[kCap];
        int nd = 0;
        const WinRanges rD = k2_win_ranges(Rd, VD, h.x, h.y, wyD, wzD);
        const WinRanges rU = k2_win_ranges(Ru, VU, h.x, h.y, wyU, wzU);
        k2_scan(rD, Rd, VD, [&](int k, float2 c) {
            if (fabsf(c.x - h.x) <= wyD && fabsf(c.y - h.y) <= wzD) {
                if (nd < kCap) { cy[nd] = wd * c.x; cz[nd] = wd * c.y; ck[nd] = k; }
                nd++;
            }
        });
        int bestU = -1, bestD = -1;
        float best = 0.0f;
        auto consider = [&](int ku, int kd, float d2) {
            bool better = bestU < 0 || d2 < best;
            if (!better && d2 == best) {   // exact tie: smaller load index of u, then of d
                const uint32_t ou = origU[ku], ob = origU[bestU];
                better = ou < ob || (ou == ob && origD[kd] < origD[bestD]);
            }
            if (better) { best = d2; bestU = ku; bestD = kd; }
        };
        if (nd > 0) {
            k2_scan(rU, Ru, VU, [&](int ku, float2 c) {
                if (!(fabsf(c.x - h.x) <= wyU && fabsf(c.y - h.y) <= wzU)) return;
                const float py = wu * c.x, pz = wu * c.y;
                if (nd <= kCap) {
                    for (int j = 0; j < nd; j++) {
                        const float ey = h.x - (py + cy[j]), ez = h.y - (pz + cz[j]);
                        consider(ku, ck[j], ey * ey + ez * ez);
                    }
                } else {
                    // More down-candidates than the cache holds (dense rows: time frames).  A pair counts only if its
                    // residual is <= nf_d2max, i.e. if the down-hit lies within sqrt(nf_d2max) / wd of the point that
                    // this up-hit mirrors through h; so the down row's grid is asked for that box (with a margin far
                    // above the rounding of the two expressions) instead of the whole window again: the pairs left
                    // out are rejected whatever their order, the others are compared exactly as before.
                    const float my = (h.x - py) * rwd, mz = (h.y - pz) * rwd;
                    // (the box cut to the window: what a staged block holds of the row is what the window can reach)
                    k2_for_box(Rd, VD, fmaxf(my - boxR, h.x - wyD), fminf(my + boxR, h.x + wyD), fmaxf(mz - boxR, h.y - wzD),
                               fminf(mz + boxR, h.y + wzD), [&](int kd, float2 e) {
                        if (!(fabsf(e.x - h.x) <= wyD && fabsf(e.y - h.y) <= wzD)) return;
                        const float ey = h.x - (py + wd * e.x), ez = h.y - (pz + wd * e.y);
                        consider(ku, kd, ey * ey + ez * ez);
                    });
                }
            });
        }
        const bool ok = bestU >= 0 && best <= dp.P.nf_d2max;
        up[i] = ok ? bestU : -1;
        dn[i] = ok ? bestD : -1;
    }
}

// ------------------------------------------------------------------------------------------ K3 + K4
// Cleaner (S3): keep reciprocal links only.  Start hits (S4): no down-link, chain of >= seed_min_chain hits.
// The chain test re-derives the cleaned up-links of the next rows from the raw links (same predicate), so one
// kernel does both; the start lists are appended with one atomic per block (collected in shared memory).
#ifndef TPC_K3T
#define TPC_K3T 64
#endif
constexpr int kK3Threads = TPC_K3T;


__device__ __forceinline__ int clean_up_link(const DevPtrs& d, int hitOff, int hitOffUp, int i) {
    const int u = d.linkUp[hitOff + i];
    return (u >= 0 && d.linkDn[hitOffUp + u] == i) ? u : -1;
}

constexpr int kK3Buf = 512;    // start hits a block collects in shared memory before it appends them (8 KB)
static_assert(kK3Buf % kK3Threads == 0, "K3 empties its buffer on iteration boundaries");

__global__ void __launch_bounds__(kK3Threads) k3_clean_start(DevPtrs d, DevParams dp, int sectorMajor) {
    grid_dep_wait();
#if TPC_PDL_TRIGGER
    grid_dep_trigger();      // K5 may stage its row table (written by K1) while this kernel runs out
#endif
    // Blocks run pad row by pad row (all sectors of row 0, then row 1, ...): blocks are dispatched in index order, so
    // the start list comes out roughly ordered by pad row.  K5 gives 32 consecutive start hits to a warp; tracklets
    // that start in the same row are in the same leg at the same time far more often than random ones, so the lanes
    // of a warp finish together (fewer half-empty warp steps).  Nothing depends on the order.
    // sectorMajor (time frames: thousands of tracklets per sector): one sector's rows after the other, so that the
    // tracklets the free-running K5 kernel has in flight at a time share a sector's hits and buckets in L2
    // (time frame: K5 23.9 -> 21.8 ms, K6 5.3 -> 4.3 ms; with 4 central events per call it costs 12 %, hence the switch)
    const int r = sectorMajor ? (int)blockIdx.x % dp.nRows : (int)blockIdx.x / dp.nSec;
    const int rowId = sectorMajor ? (int)blockIdx.x : ((int)blockIdx.x - r * dp.nSec) * dp.nRows + r;
    const int n = d.meta[rowId].n;
    if (n == 0) return;
    // The block's start hits are collected in shared memory and appended with ONE atomic per list and block: with
    // an atomic per warp and 64 hits, half of the kernel's time was spent waiting in line at counters[kNStart].
    __shared__ int4 sStart[kK3Buf];
    __shared__ unsigned sCount, sBaseRaw, sBaseRow, sStored;
    if (threadIdx.x == 0) sCount = 0u;
    __syncthreads();
    auto flush = [&]() {      // called by all threads
        __syncthreads();
        const unsigned cnt = sCount;
        if (cnt == 0u) return;
        if (threadIdx.x == 0) {
            const unsigned raw = atomicAdd(&d.counters[kNStart], cnt);
            const unsigned room = raw < (unsigned)d.maxTracklets ? (unsigned)d.maxTracklets - raw : 0u;
            const unsigned nst = min(cnt, room);
            sBaseRaw = raw; sStored = nst;
            sBaseRow = nst ? atomicAdd(&d.rowHist[r], nst) : 0u;     // ... and filed under its pad row (phased K5)
        }
        __syncthreads();
        const unsigned nst = sStored, b0 = sBaseRaw, b1 = d.rowStartBase[r] + sBaseRow;
        for (unsigned k = threadIdx.x; k < nst; k += kK3Threads) {
            const int4 v = sStart[k];
            d.startsRaw[b0 + k] = v;
            d.starts[b1 + k] = v;
        }
        __syncthreads();
        if (threadIdx.x == 0) sCount = 0u;
        __syncthreads();
    };
    const bool hasUp = r + 1 < dp.nRows, hasDn = r >= 1;
    const int hitOff = d.grid[rowId].hitOff;
    const int hitOffU = hasUp ? d.grid[rowId + 1].hitOff : hitOff;
    const int hitOffD = hasDn ? d.grid[rowId - 1].hitOff : hitOff;
    const unsigned lane = threadIdx.x & 31u;
    unsigned nLinks = 0;
    for (int base = 0; base < n; base += kK3Threads) {
        const int i = base + threadIdx.x;
        bool isStart = false;
        int upKeep = -1;
        if (i < n) {
            const int u = d.linkUp[hitOff + i], dnl = d.linkDn[hitOff + i];
            const int uc = (u >= 0 && d.linkDn[hitOffU + u] == i) ? u : -1;
            const int dc = (dnl >= 0 && d.linkUp[hitOffD + dnl] == i) ? dnl : -1;
            d.linkUpC[hitOff + i] = uc;
            upKeep = uc;
            d.linkDnC[hitOff + i] = dc;
            nLinks += uc >= 0;
            if (dc < 0 && uc >= 0) {
                int len = 2, cur = uc, row = rowId + 1;
                while (len < dp.P.seed_min_chain && (row % dp.nRows) + 1 < dp.nRows) {
                    const int nx = clean_up_link(d, d.grid[row].hitOff, d.grid[row + 1].hitOff, cur);
                    if (nx < 0) break;
                    cur = nx; row++; len++;
                }
                isStart = len >= dp.P.seed_min_chain;
            }
        }
        // rows with more hits than the buffer holds empty it every kK3Buf hits (uniform: base is the block's)
        if (base > 0 && base % kK3Buf == 0) flush();
        const unsigned m = __ballot_sync(0xffffffffu, isStart);
        if (m) {
            unsigned pos = 0;
            if (lane == 0) pos = atomicAdd(&sCount, (unsigned)__popc(m));
            pos = __shfl_sync(0xffffffffu, pos, 0) + __popc(m & ((1u << lane) - 1u));
            if (isStart)   // (row, hit, linked hit, canonical id): all K5 needs to begin
                sStart[pos] = make_int4(rowId, i, upKeep, (int)d.orig[hitOff + i]);
        }
    }
    flush();
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) nLinks += __shfl_xor_sync(0xffffffffu, nLinks, o);
    if (lane == 0 && nLinks) atomicAdd(&d.counters[kNLinks], nLinks);
}

}  // namespace tpc
