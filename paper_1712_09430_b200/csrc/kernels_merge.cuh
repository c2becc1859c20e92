// K7 track merging (Phase II, first step): "merges track segments inside the sector for the case that there is a gap
// which the track following did not cover ... track parameters at the border of the sectors are compared and matching
// tracks are merged" (Table 1: "Matching Covariance").  Reading S7 of DESIGN.md: a segment A is continued
// outward by the segment B - same TPC side, same or neighbouring sector, first row of B above the last row of A by at
// most merge_max_row_gap - whose state is nearest in chi2 (5 parameters, summed covariances) once A's state has been
// rotated into B's sector frame and propagated to B's reference x; the link is kept if it is mutual.
// One thread per segment; the candidates of a segment are contiguous in a list of the tracks ordered by
// (sector, first row), which three small kernels build first.  -fmad=false: every product and sum below is the IEEE
// fp32 operation written (the oracle evaluates the same expressions in the same order).
#pragma once
#include "kernels_kf.cuh"

namespace tpc {

struct MergePtrs {
    const tpc_track* tracks;       // K6b's output
    const uint32_t* clusterIds;
    const uint32_t* counters;      // counters[kNTracks]
    uint32_t* key;                 // canonical id of a track: its first cluster id
    uint32_t* binStart;            // [nSec * nRows + 2] tracks per (sector, first row), then its exclusive prefix
    uint32_t* binCursor;           // [nSec * nRows + 1]
    uint32_t* order;               // track indices ordered by (sector, first row)
    unsigned long long* bestIn;    // per track: min over inner partners of (chi2 bits << 32 | key of the partner)
    int32_t* out;                  // per track: best outer partner, -1 none
    float* outChi2;
    int32_t* next;                 // mutual links
    int32_t* prev;
    float* chi2;                   // chi2 of the link i -> next[i]
    tpc_merged_track* merged;
    int32_t* segments;
    uint32_t* mcount;              // [0] merged tracks, [1] segments written (one 64-bit word)
    int32_t nBins;                 // nSec * nRows
};

constexpr int kK7Threads = 128;

__global__ void __launch_bounds__(kK7Threads) k7_init(MergePtrs m, int nRows) {
    grid_dep_wait();
    const unsigned nT = m.counters[kNTracks];
    const unsigned i = blockIdx.x * kK7Threads + threadIdx.x;
    const unsigned stride = gridDim.x * kK7Threads;
    for (unsigned b = i; b <= (unsigned)m.nBins + 1u; b += stride) { m.binStart[b] = 0u; if (b <= (unsigned)m.nBins) m.binCursor[b] = 0u; }
    if (i == 0) { m.mcount[0] = 0u; m.mcount[1] = 0u; }
    for (unsigned t = i; t < nT; t += stride) {
        m.bestIn[t] = ~0ull; m.out[t] = -1; m.next[t] = -1; m.prev[t] = -1; m.chi2[t] = 0.f; m.outChi2[t] = 0.f;
        m.key[t] = m.clusterIds[m.tracks[t].cluster_offset];
    }
}
__global__ void __launch_bounds__(kK7Threads) k7_hist(MergePtrs m, int nRows) {
    grid_dep_wait();
    const unsigned nT = m.counters[kNTracks];
    for (unsigned t = blockIdx.x * kK7Threads + threadIdx.x; t < nT; t += gridDim.x * kK7Threads)
        atomicAdd(&m.binStart[m.tracks[t].sector * nRows + m.tracks[t].first_row], 1u);
}
// exclusive prefix of binStart[0..nBins] in place (one block; nBins is a few thousand)
__global__ void __launch_bounds__(1024) k7_scan(MergePtrs m) {
    grid_dep_wait();
    __shared__ uint32_t warpSum[32];
    __shared__ uint32_t carry;
    if (threadIdx.x == 0) carry = 0u;
    __syncthreads();
    for (int base = 0; base <= m.nBins; base += 1024) {
        const int b = base + threadIdx.x;
        const uint32_t v = b <= m.nBins ? m.binStart[b] : 0u;
        uint32_t incl = v;
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) {
            const uint32_t u = __shfl_up_sync(0xffffffffu, incl, o);
            if ((threadIdx.x & 31) >= o) incl += u;
        }
        if ((threadIdx.x & 31) == 31) warpSum[threadIdx.x >> 5] = incl;
        __syncthreads();
        uint32_t off = carry;
        for (int w = 0; w < (int)(threadIdx.x >> 5); w++) off += warpSum[w];
        if (b <= m.nBins) m.binStart[b] = off + incl - v;
        __syncthreads();
        if (threadIdx.x == 1023) carry = off + incl;
        __syncthreads();
    }
    if (threadIdx.x == 0) m.binStart[m.nBins + 1] = carry;
}
__global__ void __launch_bounds__(kK7Threads) k7_scatter(MergePtrs m, int nRows) {
    grid_dep_wait();
    const unsigned nT = m.counters[kNTracks];
    for (unsigned t = blockIdx.x * kK7Threads + threadIdx.x; t < nT; t += gridDim.x * kK7Threads) {
        const int b = m.tracks[t].sector * nRows + m.tracks[t].first_row;
        m.order[m.binStart[b] + atomicAdd(&m.binCursor[b], 1u)] = t;      // (order inside a bin: no result depends on it)
    }
}

// The state in a frame rotated by +beta about z, at the plane x' = const through its own point (S7); cb, sb = cos/sin
// beta.  false: the track does not move along the new x.  C' = J C J^T, J = identity except
// J00 = c/c', J10 = -t sb/c', J20 = -k CB sb, J22 = c'/c; sums in ascending index order.
__device__ __forceinline__ bool k7_rotate(KFState& a, float& x, float cb, float sb, float CB, float smax) {
    const float y = a.p0, s = a.p2, t = a.p3, k = a.p4;
    const float c = sqrtf(1.0f - s * s);
    const float s2 = s * cb - c * sb;
    const float c2 = c * cb + s * sb;
    if (!(c2 > 0.f) || !(fabsf(s2) < smax) || !(fabsf(s) < smax)) return false;
    const float J00 = c / c2, J10 = -(t * sb) / c2, J20 = -((k * CB) * sb), J22 = c2 / c;
    // full symmetric C: C[i][j], i >= j -> lower-triangle index
    const float C00 = a.c0, C10 = a.c1, C11 = a.c2, C20 = a.c3, C21 = a.c4, C22 = a.c5, C30 = a.c6, C31 = a.c7, C32 = a.c8,
                C33 = a.c9, C40 = a.c10, C41 = a.c11, C42 = a.c12, C43 = a.c13, C44 = a.c14;
    // A = J C (rows 0..2; rows 3, 4 are C's)
    const float A00 = J00 * C00, A01 = J00 * C10, A02 = J00 * C20, A03 = J00 * C30, A04 = J00 * C40;
    const float A10 = J10 * C00 + C10, A11 = J10 * C10 + C11, A12 = J10 * C20 + C21, A13 = J10 * C30 + C31, A14 = J10 * C40 + C41;
    const float A20 = J20 * C00 + J22 * C20, A21 = J20 * C10 + J22 * C21, A22 = J20 * C20 + J22 * C22,
                A23 = J20 * C30 + J22 * C32, A24 = J20 * C40 + J22 * C42;
    // C' = A J^T, lower triangle: column 0: *J00; column 1: A.0*J10 + A.1; column 2: A.0*J20 + A.2*J22; columns 3, 4: A.3, A.4
    a.c0 = A00 * J00;
    a.c1 = A10 * J00;              a.c2 = A10 * J10 + A11;
    a.c3 = A20 * J00;              a.c4 = A20 * J10 + A21;        a.c5 = A20 * J20 + A22 * J22;
    a.c6 = C30 * J00;              a.c7 = C30 * J10 + C31;        a.c8 = C30 * J20 + C32 * J22;   a.c9 = C33;
    a.c10 = C40 * J00;             a.c11 = C40 * J10 + C41;       a.c12 = C40 * J20 + C42 * J22;  a.c13 = C43;  a.c14 = C44;
    (void)A01; (void)A02; (void)A03; (void)A04; (void)A12; (void)A13; (void)A14; (void)A23; (void)A24;
    const float xn = x * cb + y * sb;
    a.p0 = y * cb - x * sb;
    x = xn;
    a.p2 = s2;
    return true;
}

// chi2 = d^T S^-1 d by LDL^T without pivoting (S symmetric 5x5, lower triangle s[15]); 1e30 if a pivot is not positive.
// The forward substitution w = L^-1 d runs along with the factorisation (row j needs the columns < j only), term by term
// in the order of the definition: chi2 = sum_j w_j^2 / D_j.  Every term is >= 0 while the pivots are positive, so the
// partial sums never fall: as soon as one exceeds `cap` (the caller rejects chi2 > cap) or a pivot fails, the
// candidate's fate is decided and the rest is skipped - most candidates are strangers and leave at the first term.
// A returned value <= cap is the full sum.
__device__ __forceinline__ float k7_chi2(const float d[5], const float s[15], float cap) {
    float L[5][5], D[5], w[5];
    auto S = [&](int i, int j) { return s[i * (i + 1) / 2 + j]; };      // i >= j
    float chi = 0.f;
#pragma unroll
    for (int j = 0; j < 5; j++) {
        float dj = S(j, j);
#pragma unroll
        for (int q = 0; q < j; q++) dj = dj - (L[j][q] * L[j][q]) * D[q];
        if (!(dj > 0.f)) return 1e30f;
        D[j] = dj;
        float v = d[j];
#pragma unroll
        for (int q = 0; q < j; q++) v = v - L[j][q] * w[q];
        w[j] = v;
        chi = chi + (v * v) / dj;
        if (!(chi <= cap)) return chi;
#pragma unroll
        for (int i = j + 1; i < 5; i++) {
            float u = S(i, j);
#pragma unroll
            for (int q = 0; q < j; q++) u = u - (L[i][q] * L[j][q]) * D[q];
            L[i][j] = u / dj;
        }
    }
    return chi;
}

__device__ __forceinline__ unsigned long long k7_pack(float chi2, uint32_t key) {
    return ((unsigned long long)__float_as_uint(chi2) << 32) | (unsigned long long)key;
}

// One WARP per segment A (its candidates - a few to a few dozen - are shared out over the lanes): A's best outer
// partner, and A's bid for being the best inner partner of every match.
__global__ void __launch_bounds__(kK7Threads) k7_match(MergePtrs m, DevParams dp, int perSide, float cosB, float sinB) {
    grid_dep_wait();
    const unsigned nT = m.counters[kNTracks];
    const int nRows = dp.nRows;
    const unsigned lane = threadIdx.x & 31u;
    const unsigned warp = (blockIdx.x * kK7Threads + threadIdx.x) >> 5, nWarps = (gridDim.x * kK7Threads) >> 5;
    for (unsigned a = warp; a < nT; a += nWarps) {
        const tpc_track TA = m.tracks[a];
        const int side = TA.sector / perSide, sa = TA.sector - side * perSide;
        const uint32_t keyA = m.key[a];
        const int rLo = TA.last_row + 1, rHi = min(TA.last_row + dp.P.merge_max_row_gap, nRows - 1);
        int best = -1;
        float bestC = 0.f;
        uint32_t bestKey = 0u;
        if (rLo <= rHi) {
#pragma unroll 1
            for (int ds = -1; ds <= 1; ds++) {
                // the neighbouring sectors in the ring of perSide sectors of this TPC side (1 sector: none; 2 sectors: the
                // other one, once), and the signed step -1 / 0 / +1 between the two frames
                if (ds != 0 && (perSide < 2 || (perSide == 2 && ds < 0))) continue;
                int sb = sa + ds;
                if (sb < 0) sb += perSide;
                if (sb >= perSide) sb -= perSide;
                const int secB = side * perSide + sb;
                const unsigned j0 = m.binStart[secB * nRows + rLo], j1 = m.binStart[secB * nRows + rHi + 1];
                if (j0 >= j1) continue;
                int dsec = sb - sa;
                if (dsec > perSide / 2) dsec -= perSide;
                if (dsec < -perSide / 2) dsec += perSide;
                // A's state in B's frame (the same for every candidate of this sector)
                KFState st;
                st.p0 = TA.p[0]; st.p1 = TA.p[1]; st.p2 = TA.p[2]; st.p3 = TA.p[3]; st.p4 = TA.p[4];
                st.c0 = TA.c[0]; st.c1 = TA.c[1]; st.c2 = TA.c[2]; st.c3 = TA.c[3]; st.c4 = TA.c[4]; st.c5 = TA.c[5]; st.c6 = TA.c[6];
                st.c7 = TA.c[7]; st.c8 = TA.c[8]; st.c9 = TA.c[9]; st.c10 = TA.c[10]; st.c11 = TA.c[11]; st.c12 = TA.c[12];
                st.c13 = TA.c[13]; st.c14 = TA.c[14];
                float xA = TA.x;
                if (dsec != 0 && !k7_rotate(st, xA, cosB, dsec > 0 ? sinB : -sinB, dp.CB, dp.P.kf_smax)) continue;
#pragma unroll 1
                for (unsigned j = j0 + lane; j < j1; j += 32u) {
                    const unsigned b = m.order[j];
                    if (b == a) continue;
                    const tpc_track TB = m.tracks[b];
                    KFState o;
                    if (!kf_propagate(st, TB.x - xA, dp.CB, dp.P.kf_smax, o)) continue;
                    const float d[5] = {o.p0 - TB.p[0], o.p1 - TB.p[1], o.p2 - TB.p[2], o.p3 - TB.p[3], o.p4 - TB.p[4]};
                    const float s[15] = {o.c0 + TB.c[0], o.c1 + TB.c[1], o.c2 + TB.c[2], o.c3 + TB.c[3], o.c4 + TB.c[4],
                                         o.c5 + TB.c[5], o.c6 + TB.c[6], o.c7 + TB.c[7], o.c8 + TB.c[8], o.c9 + TB.c[9],
                                         o.c10 + TB.c[10], o.c11 + TB.c[11], o.c12 + TB.c[12], o.c13 + TB.c[13], o.c14 + TB.c[14]};
                    const float c = k7_chi2(d, s, dp.P.merge_chi2);
                    if (!(c <= dp.P.merge_chi2)) continue;
                    const uint32_t keyB = m.key[b];
                    if (best < 0 || c < bestC || (c == bestC && keyB < bestKey)) { best = (int)b; bestC = c; bestKey = keyB; }
                    atomicMin(&m.bestIn[b], k7_pack(c, keyA));
                }
            }
        }
        // the warp's best: smaller chi2, then smaller key (lanes without a match carry the largest possible word)
        unsigned long long w = best >= 0 ? k7_pack(bestC, bestKey) : ~0ull;
        int wb = best;
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) {
            const unsigned long long w2 = __shfl_xor_sync(0xffffffffu, w, o);
            const int b2 = __shfl_xor_sync(0xffffffffu, wb, o);
            if (w2 < w) { w = w2; wb = b2; }
        }
        if (lane == 0) {
            m.out[a] = wb;
            m.outChi2[a] = wb >= 0 ? __uint_as_float((unsigned)(w >> 32)) : 0.f;
        }
    }
}
// A link survives if it is mutual.
__global__ void __launch_bounds__(kK7Threads) k7_link(MergePtrs m) {
    grid_dep_wait();
    const unsigned nT = m.counters[kNTracks];
    for (unsigned a = blockIdx.x * kK7Threads + threadIdx.x; a < nT; a += gridDim.x * kK7Threads) {
        const int b = m.out[a];
        if (b >= 0 && m.bestIn[b] == k7_pack(m.outChi2[a], m.key[a])) { m.next[a] = b; m.prev[b] = (int)a; m.chi2[a] = m.outChi2[a]; }
    }
}
// Merged tracks: one per segment without inner partner, its chain written out.
__global__ void __launch_bounds__(kK7Threads) k7_chains(MergePtrs m) {
    grid_dep_wait();
    const unsigned nT = m.counters[kNTracks];
    for (unsigned h = blockIdx.x * kK7Threads + threadIdx.x; h < nT; h += gridDim.x * kK7Threads) {
        if (m.prev[h] >= 0) continue;
        int nSeg = 0, nCl = 0;
        for (int i = (int)h; i >= 0 && nSeg < (int)nT; i = m.next[i]) { nSeg++; nCl += m.tracks[i].n_clusters; }
        const unsigned long long old = atomicAdd(reinterpret_cast<unsigned long long*>(m.mcount),
                                                 ((unsigned long long)(unsigned)nSeg << 32) | 1ull);
        const unsigned slot = (unsigned)old, off = (unsigned)(old >> 32);
        tpc_merged_track r;
        r.n_segments = nSeg; r.n_clusters = nCl; r.segment_offset = (int)off; r.first_track = (int)h;
        m.merged[slot] = r;
        int k = 0;
        for (int i = (int)h; i >= 0 && k < nSeg; i = m.next[i]) m.segments[off + k++] = i;
    }
}

// ------------------------------------------------------------------------------------------ K8
// Final fit of the merged tracks (Phase II, second step, reading S8): ONE inward Kalman pass over all
// clusters of a merged track, outermost cluster first (it is the starting point), across the sector frames of its
// segments (k7_rotate); per step the curvature constant follows the field polynomial at the state's point and the
// multiple scattering over the step's path is added to the covariance.  One thread per merged track: the pass is a
// chain of up to ~450 dependent steps, so what bounds the kernel is that chain for the longest merged track.
__device__ __forceinline__ float k8_field_cb(const KFState& a, float x, float CB, float ar, float az) {
    const float r2 = x * x + a.p0 * a.p0;
    return CB * (1.0f + ar * r2 + az * (a.p1 * a.p1));
}
__device__ __forceinline__ void k8_scatter(KFState& a, float L, float x0inv) {
    const float s = a.p2, t = a.p3, k = a.p4;
    const float one_t2 = 1.0f + t * t;
    const float th2 = (0.0136f * 0.0136f) * ((k * k) / one_t2) * (L * x0inv);
    a.c5 = a.c5 + (th2 * (1.0f - s * s)) * one_t2;
    a.c9 = a.c9 + (th2 * one_t2) * one_t2;
    a.c13 = a.c13 + ((th2 * t) * k) * one_t2;
    a.c14 = a.c14 + ((th2 * t) * t) * (k * k);
}

__global__ void __launch_bounds__(kK7Threads) k8_refit(MergePtrs m, DevPtrs d, DevParams dp, tpc_refit_track* __restrict__ out,
                                                       int perSide, float cosB, float sinB) {
    const unsigned nM = m.mcount[0];
    const tpc_params& P = dp.P;
    for (unsigned i = blockIdx.x * kK7Threads + threadIdx.x; i < nM; i += gridDim.x * kK7Threads) {
        const tpc_merged_track M = m.merged[i];
        const int32_t* segs = m.segments + M.segment_offset;
        const tpc_track inner = m.tracks[segs[0]];
        const tpc_track outer = m.tracks[segs[M.n_segments - 1]];
        KFState st;
        st.p0 = outer.p[0]; st.p1 = outer.p[1]; st.p2 = outer.p[2]; st.p3 = outer.p[3]; st.p4 = outer.p[4];
        st.c0 = st.c1 = st.c2 = st.c3 = st.c4 = st.c5 = st.c6 = st.c7 = st.c8 = st.c9 = st.c10 = st.c11 = st.c12 = st.c13 = st.c14 = 0.f;
        float x = outer.x, chi2 = 0.f;
        int nfit = 0, curSector = outer.sector;
        KFState nw;
        bool ok = kf_propagate(st, d.rowX[outer.last_row] - x, k8_field_cb(st, x, dp.CB, P.field_ar, P.field_az), P.kf_smax, nw);
        if (ok) st = nw;
        bool first = true;
        // The clusters of the merged track, outermost first: segment after segment inward, each from its last cluster to
        // its first.  The pass is a chain of dependent steps, so what a step reads is requested ahead of it: the
        // cluster's sorted position and pad row two steps ahead (qPos, qRow), its coordinates and the row's x one step
        // ahead (nH, nX) - otherwise every step would wait for two dependent memory round trips.
        const int nSteps = M.n_clusters;          // = sum of the segments' clusters (k7_chains)
        int qSg = M.n_segments - 1, qOff = outer.cluster_offset, qC = outer.n_clusters - 1, qSector = outer.sector;
        auto q_next = [&]() {                     // the cursor moves one cluster inward
            if (qC > 0) { qC--; return; }
            qSg--;
            const tpc_track* tn = m.tracks + segs[qSg];
            qOff = tn->cluster_offset; qC = tn->n_clusters - 1; qSector = tn->sector;
        };
        uint32_t qPos = d.clusterPos[(unsigned)qOff + (unsigned)qC];
        int qRow = d.clusterRow[(unsigned)qOff + (unsigned)qC], qSec = qSector;
        float2 nH = d.hits[qPos];
        float nX = d.rowX[qRow];
        int nSec = qSec;
        if (nSteps > 1) { q_next(); qPos = d.clusterPos[(unsigned)qOff + (unsigned)qC]; qRow = d.clusterRow[(unsigned)qOff + (unsigned)qC]; qSec = qSector; }
        for (int k = 0; ok && k < nSteps; k++) {
            const float2 h = nH;
            const float xr = nX;
            const int sec = nSec;
            if (k + 1 < nSteps) { nH = d.hits[qPos]; nX = d.rowX[qRow]; nSec = qSec; }
            if (k + 2 < nSteps) { q_next(); qPos = d.clusterPos[(unsigned)qOff + (unsigned)qC]; qRow = d.clusterRow[(unsigned)qOff + (unsigned)qC]; qSec = qSector; }
            if (first) {           // the outermost cluster is the starting point, not a measurement
                st.p0 = h.x; st.p1 = h.y; x = xr;
                kf_init_cov(st, P);
                chi2 = 0.f; nfit = 0;
                first = false;
                continue;
            }
            if (sec != curSector) {       // into the next segment's sector frame
                int dsec = sec % perSide - curSector % perSide;
                if (dsec > perSide / 2) dsec -= perSide;
                if (dsec < -perSide / 2) dsec += perSide;
                ok = k7_rotate(st, x, cosB, dsec > 0 ? sinB : -sinB, k8_field_cb(st, x, dp.CB, P.field_ar, P.field_az), P.kf_smax);
                curSector = sec;
                if (!ok) break;
            }
            const float x0 = x, y0 = st.p0, z0 = st.p1;
            ok = kf_propagate(st, xr - x, k8_field_cb(st, x, dp.CB, P.field_ar, P.field_az), P.kf_smax, nw);
            if (!ok) break;
            st = nw; x = xr;
            if (P.ms_x0_inv > 0.f) {
                const float dx = x - x0, dy = st.p0 - y0, dz = st.p1 - z0;
                k8_scatter(st, sqrtf((dx * dx + dy * dy) + dz * dz), P.ms_x0_inv);
            }
            kf_update_hit(st, h.x, h.y, P.err2_y, P.err2_z, chi2, true);
            nfit++;
        }
        tpc_refit_track r;
        r.first_track = segs[0];
        if (ok && !first) {
            r.sector = curSector; r.n_fit = nfit; r.ok = 1; r.x = x; r.chi2 = chi2;
            r.p[0] = st.p0; r.p[1] = st.p1; r.p[2] = st.p2; r.p[3] = st.p3; r.p[4] = st.p4;
            r.c[0] = st.c0; r.c[1] = st.c1; r.c[2] = st.c2; r.c[3] = st.c3; r.c[4] = st.c4; r.c[5] = st.c5; r.c[6] = st.c6; r.c[7] = st.c7;
            r.c[8] = st.c8; r.c[9] = st.c9; r.c[10] = st.c10; r.c[11] = st.c11; r.c[12] = st.c12; r.c[13] = st.c13; r.c[14] = st.c14;
        } else {                       // the pass could not be completed: the innermost segment's Phase-I state
            r.sector = inner.sector; r.n_fit = 0; r.ok = 0; r.x = inner.x; r.chi2 = inner.chi2;
#pragma unroll
            for (int q = 0; q < 5; q++) r.p[q] = inner.p[q];
#pragma unroll
            for (int q = 0; q < 15; q++) r.c[q] = inner.c[q];
        }
        out[i] = r;
    }
}

}  // namespace tpc
