// K5 tracklet constructor, pooled form: ONE persistent kernel for any number of tracklets.
//
// "varying track length" limits vectorisation and GPU utilisation, "insufficient tracks per sector".
// With one thread per track candidate a warp lasts as long as its longest tracklet in every leg, and
// measured on a central event the lanes of the warp-phased kernel were 40 % idle (ncu r01h: 19.1 of 32 threads per
// instruction; modelled from the oracle's tracklets: 173 M warp instructions against 104 M with perfect packing).
// Here a tracklet is not tied to a thread: its filter state lives in a 160-byte record in global memory (L2) and is
// in registers only for a SLICE of pad-row steps.  Each SM (one block) keeps three queues of tracklets in shared
// memory, one per kind of work,
//     HEAVY  legs A (follow the seed's links), B (extrapolate outward) and D (extend inward below the seed):
//            the full step with road search
//     LIGHT  leg C (filter inward over the hits found): propagate + update, no search
//     DONE   tracklet complete: first pass of the selector (S6) over its hits, warp-wide, a pad row per lane
// and every warp repeats: take up to 32 tracklets of the fullest queue, load their states, run that kind's loop for
// a slice (until kSlice steps are done or a quarter of the lanes have left the leg), store the states and file each
// tracklet under the kind of its next leg.  Warps therefore run full whatever the lengths of the tracklets are, every
// step is the cheapest one for its leg, and the same kernel serves one event (all tracklets of the SM in flight at
// once) and time frames (new groups of 32 start hits are admitted while fewer than kMaxLive tracklets are live).
// The arithmetic of a step is kernels_kf.cuh's (kf_propagate, kf_update_hit, road_search_fast), unchanged: which
// thread evaluates a step does not enter any result.
#pragma once
#include "kernels_kf.cuh"

namespace tpc {

#ifndef TPC_K5P_SLICE
#define TPC_K5P_SLICE 16
#endif
#ifndef TPC_K5P_MINBATCH
#define TPC_K5P_MINBATCH 1
#endif
#ifndef TPC_K5P_MINSTEPS
#define TPC_K5P_MINSTEPS 4
#endif
constexpr int kK5PoolThreads = 384;
constexpr int kK5PoolWarps = kK5PoolThreads / 32;
constexpr int kSlice = TPC_K5P_SLICE;          // pad-row steps per slice at most
constexpr int kSliceMin = TPC_K5P_MINSTEPS;    // ... and at least (unless every lane has left the leg)
constexpr int kRing = 1024;                    // queue capacity (power of two), > kMaxLive + DONE backlog + one push per warp
constexpr int kMaxLive = 512;                  // tracklets begun and not complete, per SM
constexpr int kDoneUrgent = 256;               // DONE backlog at which the weights pass goes first
enum : int { kQHeavy = 0, kQLight = 1, kQDone = 2, kNQ = 3, kQNew = 3, kQNone = 4 };

// Filter state of a tracklet between slices (global memory; 10 x 16 bytes).
struct __align__(16) TrackletLive {
    float p[5];
    float c[15];
    float chi2, yTop, zTop, sTop;
    float tTop, kTop, slopeY, slopeZ;
    float roadY, roadZ;
    int32_t idxC, hitAtR;
    int32_t hBelowTop;
    uint32_t startGid;
    int32_t rowBase;
    uint32_t packA;        // r | r0 << 8 | rTop << 16 | firstRow << 24
    uint32_t packB;        // (rr + 1) | nHits << 16 | nfit << 24
    uint32_t packC;        // gap | leg << 8 | lastUpd << 16
    uint32_t pad[2];
};
static_assert(sizeof(TrackletLive) == 160, "TrackletLive layout");

struct K5PoolShared {
    uint32_t ring[kNQ][kRing];
    uint32_t head[kNQ], tail[kNQ];      // monotonic; entries [head, tail) are valid
    uint32_t lock;
    uint32_t busy;                      // warps that hold a batch of tracklets right now
    uint32_t live;                      // tracklets begun and not complete
    uint32_t newNext, newGroups;        // next group of 32 start hits of this SM / how many it has
};

__device__ __forceinline__ void k5p_lock(K5PoolShared& S) {
    while (atomicCAS(&S.lock, 0u, 1u) != 0u) __nanosleep(64);
    __threadfence_block();
}
__device__ __forceinline__ void k5p_unlock(K5PoolShared& S) {
    __threadfence_block();
    atomicExch(&S.lock, 0u);
}

template <bool kGridInSmem>
__global__ void __launch_bounds__(kK5PoolThreads, 1) k5_construct_pool(DevPtrs d, DevParams dp, TrackletLive* __restrict__ liveBuf) {
    extern __shared__ __align__(32) unsigned char k5Smem[];
    __shared__ float sRowX[kMaxRows + 1];
    __shared__ uint32_t sCum[kMaxRows + 2], sSeg[kMaxRows + 2], sWarpSum[kK5PoolWarps];
    __shared__ K5PoolShared S;
    constexpr int kT = kK5PoolThreads;
    const unsigned FULL = 0xffffffffu;
    // Prologue that needs nothing of K3/K4 (the row table is K1's): runs while K3's last blocks finish when this
    // kernel was launched as K3's programmatic dependent.
    const RowGrid* __restrict__ grid = d.grid;
    if (kGridInSmem) {
        uint4* dst = reinterpret_cast<uint4*>(k5Smem);
        const uint4* src = reinterpret_cast<const uint4*>(d.grid);
        for (int i = threadIdx.x; i < d.nRowsTotal * 2; i += kT) dst[i] = __ldcg(src + i);
        grid = reinterpret_cast<const RowGrid*>(k5Smem);
    }
    for (int i = threadIdx.x; i < dp.nRows; i += kT) sRowX[i] = d.rowX[i];
    if (threadIdx.x < kNQ) { S.head[threadIdx.x] = 0u; S.tail[threadIdx.x] = 0u; }
    grid_dep_wait();
    const unsigned nTotal = min(d.counters[kNStart], (unsigned)d.maxTracklets);
    const unsigned nGroups = (nTotal + 31u) / 32u;
    if (threadIdx.x == 0) {
        S.lock = 0u; S.live = 0u; S.newNext = 0u; S.busy = 0u;
        S.newGroups = nGroups > blockIdx.x ? (nGroups - blockIdx.x + gridDim.x - 1u) / gridDim.x : 0u;
    }
    // start hits are filed by pad row (K3/K4): sCum = exclusive prefix of the per-row counts, so that start hit number
    // `slot` in row order is record slot - sCum[r] of row r's segment (r by binary search in begin())
    {
        const unsigned tid = threadIdx.x, ln = tid & 31u;
        const uint32_t h = (int)tid < dp.nRows ? d.rowHist[tid] : 0u;
        uint32_t incl = h;
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) {
            const uint32_t v = __shfl_up_sync(FULL, incl, o);
            if (ln >= (unsigned)o) incl += v;
        }
        if (ln == 31) sWarpSum[tid >> 5] = incl;
        __syncthreads();
        uint32_t off = 0;
        for (unsigned w = 0; w < (tid >> 5); w++) off += sWarpSum[w];
        if (tid <= kMaxRows + 1) sCum[tid] = off + incl - h;
        if ((int)tid <= dp.nRows) sSeg[tid] = d.rowStartBase[tid];
    }
    __syncthreads();
    const tpc_params& P = dp.P;
    const int nRows = dp.nRows;
    const unsigned lane = threadIdx.x & 31u;

    // ---- the tracklet in this lane's registers
    int leg = kLegIdle;
    int rowBase = 0, r0 = 0, r = 0, rr = 0, idxC = -1, nHits = 0, gap = 0, nfit = 0, firstRow = 0, rTop = 0;
    int hitAtR = -1, hBelowTop = -1;
    float yTop = 0.f, zTop = 0.f, sTop = 0.f, tTop = 0.f, kTop = 0.f, chi2 = 0.f;
    float slopeY = 0.f, slopeZ = 0.f;
    bool lastUpd = true;
    uint32_t startGid = 0;
    KFState st;
    unsigned slot = 0;
    int32_t* rh = d.rowHit;
    TrackletRec* rec = d.recs;
    float2 hk = make_float2(0.f, 0.f);
    int idxNraw = -1;
    Bucket B00, B01, B10, B11;
    int ly0 = 0, ly1 = 0, lz0 = 0, lz1 = 0;
    float roadY = 0.5f, roadZ = 0.5f;

    // A value that arrives by a load passes through one ALU instruction (xor with a zero the compiler cannot fold) before
    // it becomes loop-carried state.  Otherwise the first instruction of EVERY step that reads such a register carries
    // the scoreboard wait of the load that may have written it on the way into the loop - and the prefetch loads
    // issued at the end of the previous step share that scoreboard, so every step waited for its own prefetch
    // (ncu: 21 % of the samples at the two loop heads, stall_long_scoreboard).
    const int zr = dp.nRows >> 30;
    auto ldf = [&](float v) { return __int_as_float(__float_as_int(v) ^ zr); };
    auto ldi = [&](int v) { return v ^ zr; };

    auto kind_of = [&](int l) { return l == kLegC ? kQLight : l == kLegIdle ? kQDone : kQHeavy; };

    // Take tracklet `s`: initial state from the first link of the seed (S5 step 1).
    auto begin = [&](unsigned s) {
        int lo = 0, hi = nRows;
        while (hi - lo > 1) {
            const int mid = (lo + hi) >> 1;
            if (sCum[mid] <= s) lo = mid; else hi = mid;
        }
        const int4 sh = d.starts[sSeg[lo] + (s - sCum[lo])];
        const int rowId = ldi(sh.x), h0 = ldi(sh.y), h1 = ldi(sh.z);
        rowBase = (rowId / nRows) * nRows;
        r0 = rowId - rowBase;
        const int off0 = grid[rowId].hitOff, off1 = grid[rowId + 1].hitOff;
        float2 a = d.hits[off0 + h0], b = d.hits[off1 + h1];
        a.x = ldf(a.x); a.y = ldf(a.y); b.x = ldf(b.x); b.y = ldf(b.y);
        startGid = (uint32_t)ldi(sh.w);
        const float dx = sRowX[r0 + 1] - sRowX[r0];
        const float dy = b.x - a.x, dz = b.y - a.y;
        const float l = __fsqrt_rn(dx * dx + dy * dy);
        st.p0 = a.x; st.p1 = a.y; st.p2 = dy / l; st.p3 = dz / l; st.p4 = 0.f;
        kf_init_cov(st, P);
        chi2 = 0.f;
        slot = s;
        rh = d.rowHit + (size_t)s * d.rhStride;
        rec = d.recs + s;
        rh[r0] = off0 + h0;
        nHits = 1; r = r0; rTop = r0; yTop = a.x; zTop = a.y; hitAtR = off0 + h0; hBelowTop = -1;
        sTop = st.p2; tTop = st.p3; kTop = st.p4;
        slopeY = __fdividef(dy, dx); slopeZ = __fdividef(dz, dx);
        idxC = h1; rr = r0 + 1;
        leg = kLegA; gap = 0; nfit = 0; firstRow = r0; lastUpd = true;
        roadY = 0.5f; roadZ = 0.5f;
    };
    auto load_live = [&](unsigned s) {
        const float4* q = reinterpret_cast<const float4*>(liveBuf + s);
        const float4 a0 = __ldcg(q + 0), a1 = __ldcg(q + 1), a2 = __ldcg(q + 2), a3 = __ldcg(q + 3), a4 = __ldcg(q + 4);
        const float4 a5 = __ldcg(q + 5), a6 = __ldcg(q + 6), a7 = __ldcg(q + 7), a8 = __ldcg(q + 8);
        st.p0 = ldf(a0.x); st.p1 = ldf(a0.y); st.p2 = ldf(a0.z); st.p3 = ldf(a0.w);
        st.p4 = ldf(a1.x); st.c0 = ldf(a1.y); st.c1 = ldf(a1.z); st.c2 = ldf(a1.w);
        st.c3 = ldf(a2.x); st.c4 = ldf(a2.y); st.c5 = ldf(a2.z); st.c6 = ldf(a2.w);
        st.c7 = ldf(a3.x); st.c8 = ldf(a3.y); st.c9 = ldf(a3.z); st.c10 = ldf(a3.w);
        st.c11 = ldf(a4.x); st.c12 = ldf(a4.y); st.c13 = ldf(a4.z); st.c14 = ldf(a4.w);
        chi2 = ldf(a5.x); yTop = ldf(a5.y); zTop = ldf(a5.z); sTop = ldf(a5.w);
        tTop = ldf(a6.x); kTop = ldf(a6.y); slopeY = ldf(a6.z); slopeZ = ldf(a6.w);
        roadY = ldf(a7.x); roadZ = ldf(a7.y); idxC = ldi(__float_as_int(a7.z)); hitAtR = ldi(__float_as_int(a7.w));
        hBelowTop = ldi(__float_as_int(a8.x)); startGid = (uint32_t)ldi(__float_as_int(a8.y)); rowBase = ldi(__float_as_int(a8.z));
        const uint32_t pa = __float_as_uint(a8.w);
        const uint2 pbc = __ldcg(reinterpret_cast<const uint2*>(q + 9));
        r = pa & 255u; r0 = (pa >> 8) & 255u; rTop = (pa >> 16) & 255u; firstRow = pa >> 24;
        rr = (int)(pbc.x & 0xffffu) - 1; nHits = (pbc.x >> 16) & 255u; nfit = pbc.x >> 24;
        gap = pbc.y & 255u; leg = (pbc.y >> 8) & 255u; lastUpd = (pbc.y >> 16) & 1u;
        slot = s;
        rh = d.rowHit + (size_t)s * d.rhStride;
        rec = d.recs + s;
    };
    auto store_live = [&]() {
        float4* q = reinterpret_cast<float4*>(liveBuf + slot);
        __stcg(q + 0, make_float4(st.p0, st.p1, st.p2, st.p3));
        __stcg(q + 1, make_float4(st.p4, st.c0, st.c1, st.c2));
        __stcg(q + 2, make_float4(st.c3, st.c4, st.c5, st.c6));
        __stcg(q + 3, make_float4(st.c7, st.c8, st.c9, st.c10));
        __stcg(q + 4, make_float4(st.c11, st.c12, st.c13, st.c14));
        __stcg(q + 5, make_float4(chi2, yTop, zTop, sTop));
        __stcg(q + 6, make_float4(tTop, kTop, slopeY, slopeZ));
        __stcg(q + 7, make_float4(roadY, roadZ, __int_as_float(idxC), __int_as_float(hitAtR)));
        const uint32_t pa = (uint32_t)r | ((uint32_t)r0 << 8) | ((uint32_t)rTop << 16) | ((uint32_t)firstRow << 24);
        __stcg(q + 8, make_float4(__int_as_float(hBelowTop), __uint_as_float(startGid), __int_as_float(rowBase), __uint_as_float(pa)));
        const uint32_t pb = (uint32_t)(rr + 1) | ((uint32_t)nHits << 16) | ((uint32_t)nfit << 24);
        const uint32_t pc = (uint32_t)min(gap, 255) | ((uint32_t)leg << 8) | ((lastUpd ? 1u : 0u) << 16);
        __stcg(reinterpret_cast<uint2*>(q + 9), make_uint2(pb, pc));
    };

    // The 2x2 buckets around the predicted position (yq, zq) in row `row`, widened by the last road (half-width capped
    // at half a bin so that the window spans at most two bins per coordinate).
    auto preload = [&](int row, float yq, float zq) {
        const RowGrid Rq = grid[rowBase + row];
        const float wy = fminf(roadY * TPC_WA + TPC_WB, __fdividef(0.49f, Rq.invY));
        const float wz = fminf(roadZ * TPC_WA + TPC_WB, __fdividef(0.49f, Rq.invZ));
        ly0 = bin_of(yq - wy, Rq.y0, Rq.invY, Rq.nY); ly1 = bin_of(yq + wy, Rq.y0, Rq.invY, Rq.nY);
        lz0 = bin_of(zq - wz, Rq.z0, Rq.invZ, Rq.nZ); lz1 = bin_of(zq + wz, Rq.z0, Rq.invZ, Rq.nZ);
        const Bucket* bq = d.buckets + Rq.binOff;
        B00 = bq[lz0 * Rq.nY + ly0]; B01 = bq[lz0 * Rq.nY + ly1];
        B10 = bq[lz1 * Rq.nY + ly0]; B11 = bq[lz1 * Rq.nY + ly1];
    };
    // Memory accesses of the NEXT step that do not depend on its arithmetic: coordinates of the linked hit of row rr and
    // the link that names the hit of the row after (leg A), the buckets of the next road search (legs B, D; harmless in A).
    // Each is ONE unconditional instruction with a selected, always valid address.
    auto issue_heavy = [&]() {
        const int hitOff = grid[rowBase + rr].hitOff;
        const bool a = leg == kLegA;
        hk = d.hits[hitOff + max(idxC, 0)];
        idxNraw = d.linkUpC[hitOff + (a ? idxC : 0)];
        const float dxq = sRowX[rr] - sRowX[r];
        preload(rr, st.p0 + slopeY * dxq, st.p1 + slopeZ * dxq);
    };
    auto issue_light = [&]() {
        const int rN = rr - 1;
        const bool wN = rN >= 0 && rN >= r0;
        hk = d.hits[max(idxC, 0)];                 // leg C: idxC is a global position
        idxNraw = rh[wN ? rN : r0];
    };
    // Legs A/B are over: re-initialise at the outermost hit and filter inward (S5 step 4).
    auto turn_inward = [&]() {
        st.p0 = yTop; st.p1 = zTop; st.p2 = sTop; st.p3 = tTop; st.p4 = kTop;
        kf_init_cov(st, P);
        chi2 = 0.f; nfit = 0; r = rTop; gap = 0; lastUpd = true; firstRow = r0;
        rr = rTop - 1;                       // >= r0 - 1 >= 0
        idxC = rr >= r0 ? hBelowTop : -1;     // = rowHit[rr], kept in a register
        leg = rr >= r0 ? kLegC : kLegD;
    };
    auto finish = [&]() {
        if (lastUpd) write_state(rec, st, r, chi2, nfit);
        rec->startGid = startGid; rec->sector = rowBase / nRows; rec->startRow = r0;
        rec->nHits = nHits; rec->firstRow = firstRow; rec->lastRow = rTop;
        rec->ownerKey = owner_key(nHits, startGid, d.sectorGidBase[rowBase / nRows]);
        leg = kLegIdle;
    };

    // ---------------- legs A, B, D: one pad-row step with road search (leg A: with the linked hit instead)
    auto step_heavy = [&]() {
        const bool outward = leg != kLegD;
        const bool search = leg != kLegA;
        const int rrN = outward ? rr + 1 : rr - 1;
        const bool hasN = outward ? rrN < nRows : rrN >= 0;
        const RowGrid Rc = grid[rowBase + rr];
        const float xr = sRowX[r], xrr = sRowX[rr];
        const float yPrev = st.p0, zPrev = st.p1, dxStep = xrr - xr;
        KFState nw;
        const bool stepped = kf_propagate(st, dxStep, dp.CB, P.kf_smax, nw);
        float2 hs;
        const int found = road_search_fast(d, Rc, nw, P, search && stepped, B00, B01, B10, B11, ly0, ly1, lz0, lz1, hs,
                                           roadY, roadZ);
        const int hit = search ? found : idxC;
        const float2 hc = search ? hs : hk;
        const bool have = stepped && hit >= 0;
        // the output state of leg D is the state after the LAST update: written when a row without hit follows
        if (stepped && !outward && !have && lastUpd) write_state(rec, st, r, chi2, nfit);
        const int gpos = hit >= 0 ? Rc.hitOff + hit : -1;     // rowHit holds GLOBAL sorted positions (K6 indexes with them)
        if (stepped) { st = nw; r = rr; rh[rr] = gpos; }      // every row between the first and last hit holds a defined value
        kf_update_hit(st, hc.x, hc.y, P.err2_y, P.err2_z, chi2, have);
        bool endLeg = !stepped;
        if (stepped) {
            const float rdx = __fdividef(1.0f, dxStep);
            slopeY = (nw.p0 - yPrev) * rdx; slopeZ = (nw.p1 - zPrev) * rdx;
            gap = have ? 0 : gap + 1;
            nHits += have ? 1 : 0;
            if (have && outward) { hBelowTop = hitAtR; rTop = rr; yTop = hc.x; zTop = hc.y; sTop = st.p2; tTop = st.p3; kTop = st.p4; }
            if (!outward) {
                nfit += have ? 1 : 0;
                lastUpd = have;
                if (have) firstRow = rr;
            }
            if (outward) hitAtR = gpos;
            endLeg = gap > P.max_gap || !hasN;
            // (hit >= -1 always holds: it only ties this use of the loaded word to the end of the step)
            const int idxN = (leg == kLegA && hit >= -1) ? idxNraw : -1;
            if (leg == kLegA && idxN < 0) leg = kLegB;      // chain exhausted: extrapolate from here
            rr = rrN; idxC = idxN;
        }
        if (endLeg) {
            if (outward) turn_inward(); else finish();
        } else {
            issue_heavy();
        }
    };
    // ---------------- leg C: propagate + update with the known hit of the row; no search, no bucket, no grid access
    auto step_light = [&]() {
        const int rrN = rr - 1;
        const bool hasN = rrN >= 0;
        const bool wantN = hasN && rrN >= r0;
        const float xr = sRowX[r], xrr = sRowX[rr];
        KFState nw;
        const bool stepped = kf_propagate(st, xrr - xr, dp.CB, P.kf_smax, nw);
        const bool have = stepped && idxC >= 0;
        if (stepped && !have && lastUpd) write_state(rec, st, r, chi2, nfit);
        if (stepped) { st = nw; r = rr; }
        kf_update_hit(st, hk.x, hk.y, P.err2_y, P.err2_z, chi2, have);
        bool endLeg = !stepped;
        if (stepped) {
            nfit += have ? 1 : 0;
            lastUpd = have;
            endLeg = !hasN;
            const int idxN = (wantN && nfit >= 0) ? idxNraw : -1;     // (nfit >= 0 always: late use of the load)
            if (rrN < r0) leg = kLegD;
            rr = rrN; idxC = idxN;
        }
        if (endLeg) finish();
        else if (leg == kLegC) issue_light();
    };

    // ---------------- S6 first pass for up to 32 complete tracklets (lane i names tracklet wslot, valid if i < n):
    // hitWeight[h] = max ownership key over the kept tracklets containing h; a pad row per lane.
    unsigned w6Kept = 0, w6Hits = 0;
    auto weights_pass = [&](unsigned wslot, unsigned n) {
        const bool hadOne = lane < n;
        const TrackletRec* tr = d.recs + (hadOne ? wslot : 0u);
        const int nHits6 = __ldcg(&tr->nHits), first6 = __ldcg(&tr->firstRow), last6 = __ldcg(&tr->lastRow);
        const uint32_t myKey = __ldcg(&tr->ownerKey);
        constexpr int kC = (kMaxRows + 31) / 32;
        const int nChunks = (nRows + 31) / 32;
        constexpr int kG = TPC_W6G;
#pragma unroll 1
        for (unsigned base = 0; base < n; base += kG) {
            int h[kG][kC];
            uint32_t key[kG];
#pragma unroll
            for (int g = 0; g < kG; g++) {
                const int src = min((int)base + g, 31);
                const int nH = __shfl_sync(FULL, nHits6, src);
                const int fr = __shfl_sync(FULL, first6, src), lr = __shfl_sync(FULL, last6, src);
                const unsigned ws = __shfl_sync(FULL, wslot, src);
                key[g] = __shfl_sync(FULL, myKey, src);
                const bool on = base + g < n;
                const int32_t* rp = d.rowHit + (size_t)ws * d.rhStride;
                if (lane == 0) { w6Hits += on ? nH : 0; w6Kept += (on && nH >= P.min_hits) ? 1u : 0u; }
#pragma unroll
                for (int c = 0; c < kC; c++) {
                    const int q = c * 32 + (int)lane;
                    h[g][c] = (on && c < nChunks && q >= fr && q <= lr && nH >= P.min_hits) ? __ldcg(rp + q) : -1;
                }
            }
#pragma unroll
            for (int g = 0; g < kG; g++)
#pragma unroll
                for (int c = 0; c < kC; c++)
                    if (h[g][c] >= 0) atomicMax(&d.weight[h[g][c]], key[g]);
        }
    };

    // ---------------- the warp's life: take work, run a slice, file the tracklets again
    volatile uint32_t* vhead = S.head;
    volatile uint32_t* vtail = S.tail;
    for (;;) {
        int kind = kQNone;
        unsigned first = 0, n = 0;
        if (lane == 0) {
            // look without the lock first (same decision on a racy snapshot; taken again under the lock): an idle warp
            // must not keep the busy ones from the queues
            bool maybe;
            {
                const unsigned cH = vtail[kQHeavy] - vhead[kQHeavy], cL = vtail[kQLight] - vhead[kQLight];
                const unsigned cD = vtail[kQDone] - vhead[kQDone];
                const unsigned live = *(volatile uint32_t*)&S.live, busy = *(volatile uint32_t*)&S.busy;
                const unsigned nn = *(volatile uint32_t*)&S.newNext;
                maybe = cH + cL > 0u || cD > 0u || (nn < S.newGroups && live + 32u <= (unsigned)kMaxLive) ||
                        (live == 0u && nn >= S.newGroups);
                (void)busy;
            }
            if (maybe) {
                k5p_lock(S);
                const unsigned cH = S.tail[kQHeavy] - S.head[kQHeavy], cL = S.tail[kQLight] - S.head[kQLight];
                const unsigned cD = S.tail[kQDone] - S.head[kQDone];
                const bool newAvail = S.newNext < S.newGroups && S.live + 32u <= (unsigned)kMaxLive;
                // One event holds ~8 warps' worth of tracklets per SM: far too few to be bound by instruction issue, the
                // time is steps-in-sequence x step latency.  So the queued tracklets are shared out evenly over the warps
                // that are free right now (a warp's share, not a full batch), and new start hits are admitted while the
                // queues cannot give every free warp 32.
                const unsigned idle = (unsigned)kK5PoolWarps - S.busy;            // >= 1: this warp
                const unsigned tot = cH + cL;
                const int best = cL > cH ? kQLight : kQHeavy;
                const unsigned cB = cL > cH ? cL : cH;
                unsigned share = 0u;
                if (cD >= (unsigned)kDoneUrgent) kind = kQDone;
                else if (newAvail && tot < 32u * idle) kind = kQNew;
                else if (tot > 0u) { kind = best; share = min(32u, min(cB, max((tot + idle - 1u) / idle, (unsigned)TPC_K5P_MINBATCH))); }
                else if (cD > 0u) kind = kQDone;
                else if (S.live == 0u && S.newNext >= S.newGroups) kind = -1;      // nothing left anywhere: leave
                if (kind == kQNew) {
                    first = (blockIdx.x + S.newNext * gridDim.x) * 32u;
                    n = min(32u, nTotal - first);
                    S.newNext++;
                    S.live += n;
                    S.busy++;
                } else if (kind == kQHeavy || kind == kQLight) {
                    n = share;
                    first = S.head[kind];
                    S.head[kind] = first + n;
                    S.busy++;
                } else if (kind == kQDone) {
                    n = min(32u, cD);
                    first = S.head[kQDone];
                    S.head[kQDone] = first + n;
                }
                k5p_unlock(S);
            }
        }
        kind = __shfl_sync(FULL, kind, 0);
        first = __shfl_sync(FULL, first, 0);
        n = __shfl_sync(FULL, n, 0);
        if (kind < 0) break;
        if (kind == kQNone) { __nanosleep(2000); continue; }
        if (kind == kQDone) {
            const unsigned ws = lane < n ? S.ring[kQDone][(first + lane) & (kRing - 1)] : 0u;
            weights_pass(ws, n);
            continue;
        }
        const bool holds = lane < n;
        if (kind == kQNew) {
            if (holds) { begin(first + lane); issue_heavy(); }
            kind = kQHeavy;
        } else if (holds) {
            load_live(S.ring[kind][(first + lane) & (kRing - 1)]);
            if (kind == kQHeavy) issue_heavy(); else issue_light();
        }
        if (!holds) leg = kLegIdle;
        // the slice: at most kSlice steps; over as soon as a quarter of its lanes have left the kind (after kSliceMin)
        const unsigned quorum = (3u * n + 3u) / 4u;
        if (kind == kQHeavy) {
#pragma unroll 1
            for (int it = 0; it < kSlice; it++) {
                const bool mine = holds && (leg == kLegA || leg == kLegB || leg == kLegD);
                const unsigned m = __ballot_sync(FULL, mine);
                if (m == 0u || (it >= kSliceMin && (unsigned)__popc(m) < quorum)) break;
                if (mine) step_heavy();
            }
        } else {
#pragma unroll 1
            for (int it = 0; it < 2 * kSlice; it++) {
                const bool mine = holds && leg == kLegC;
                const unsigned m = __ballot_sync(FULL, mine);
                if (m == 0u || (it >= kSliceMin && (unsigned)__popc(m) < quorum)) break;
                if (mine) step_light();
            }
        }
        __syncwarp();
        // file the tracklets under the kind of their next leg
        const int nk = holds ? kind_of(leg) : -1;
        if (holds && nk != kQDone) store_live();
        __threadfence();                       // states, rowHit entries and records before the queue entries
        const unsigned mH = __ballot_sync(FULL, nk == kQHeavy), mL = __ballot_sync(FULL, nk == kQLight);
        const unsigned mD = __ballot_sync(FULL, nk == kQDone);
        unsigned bH = 0u, bL = 0u, bD = 0u;
        if (lane == 0) {
            k5p_lock(S);
            bH = S.tail[kQHeavy]; bL = S.tail[kQLight]; bD = S.tail[kQDone];
        }
        bH = __shfl_sync(FULL, bH, 0); bL = __shfl_sync(FULL, bL, 0); bD = __shfl_sync(FULL, bD, 0);
        {
            const unsigned myBase = nk == kQHeavy ? bH : nk == kQLight ? bL : bD;
            const unsigned myMask = nk == kQHeavy ? mH : nk == kQLight ? mL : mD;
            if (nk >= 0) S.ring[nk][(myBase + __popc(myMask & ((1u << lane) - 1u))) & (kRing - 1)] = slot;
        }
        __syncwarp();
        if (lane == 0) {
            __threadfence_block();
            S.tail[kQHeavy] = bH + __popc(mH); S.tail[kQLight] = bL + __popc(mL); S.tail[kQDone] = bD + __popc(mD);
            S.live -= __popc(mD);
            S.busy--;
            k5p_unlock(S);
        }
        __syncwarp();
    }
    if (lane == 0) {
        if (w6Kept) atomicAdd(&d.counters[kNKept], w6Kept);
        if (w6Hits) atomicAdd(&d.counters[kHitsTotal], w6Hits);
    }
}

}  // namespace tpc
