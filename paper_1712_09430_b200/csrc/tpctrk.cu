// libtpctrk.so — C ABI (include/tpctrk.h) and host logic of the B200 Phase-I TPC sector tracker.
// Every step of the hot path runs in the kernels of kernels_ca.cuh / kernels_kf.cuh; this file only lays out
// the workspace, stages input, launches K1..K6 on the caller's stream and downloads the compacted result.
// There is no CPU fallback: without a device the compute calls return TPC_E_CUDA.
#include <algorithm>
#include <cmath>
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <mutex>
#include <new>
#include <vector>

#include "device_types.cuh"
#include "kernels_ca.cuh"
#include "kernels_kf.cuh"
#include "kernels_merge.cuh"

using namespace tpc;

namespace {

constexpr size_t kAlign = 256;
inline size_t align_up(size_t v, size_t a = kAlign) { return (v + a - 1) / a * a; }

struct Layout {   // byte offsets into the workspace
    size_t inY, inZ, grid, meta, rowX, hits, orig, binStart, buckets, linkUp, linkDn, linkUpC, linkDnC, weight, starts, startsRaw, rowHist, rowStartBase, recs, rowHit,
        tracks, clusterIds, clusterPos, clusterRow, refit, counters, sectorGidBase,
        mKey, mBinStart, mBinCursor, mOrder, mBestIn, mOut, mOutChi2, mNext, mPrev, mChi2, mMerged, mSegments, mCount, total;
    int64_t hitCap, binCap, maxTracklets;
    enum : int { kMaxGuards = 64 };
    size_t guard[kMaxGuards];        // offsets of the guard zones behind the buffers
    int nGuards;
};

}  // namespace

struct tpc_tracker {
    int nSec = 0, nRows = 0, nRowsTotal = 0, rhStride = 0;
    std::vector<float> rowX;
    tpc_params P{};
    float bz = 0.f, CB = 0.f;
    cudaStream_t stream = nullptr;
    int lastCuda = 0;
    bool dependentLaunch = true;                     // tpc_set_dependent_launch
    bool kernelTiming = false, timedCall = false;   // tpc_set_kernel_timing; whether the last call recorded ev[1..5]

    // workspace
    char* ws = nullptr;
    size_t wsBytes = 0;
    int64_t maxClusters = 0;
    Layout L{};
    DevPtrs dev{};

    // loaded event (host bookkeeping)
    std::vector<int32_t> rowN, rowIn, rowCap;   // per (sector,row): count, staging offset, slots reserved at that offset
    int64_t cursor = 0;                     // next free staging slot
    int64_t nClusters = 0;
    bool finalized = false, tracked = false, fetched = false;
    float* hostY = nullptr; float* hostZ = nullptr; int64_t hostCap = 0;   // pinned mirror for host-pointer loads
    int64_t dirtyLo = 0, dirtyHi = 0;       // host-staged range not yet uploaded
    cudaEvent_t evUpload = nullptr; bool uploadPending = false;
    cudaEvent_t evTables = nullptr; bool tablesPending = false;   // upload of the host row tables of the last finalize
    cudaEvent_t evDone = nullptr;           // after the result download queued behind K6 (tpc_track_sectors)
    int64_t estTracks = 0, estIds = 0;      // size of the download that is queued before the counts are known
    int64_t queuedTracks = 0, queuedIds = 0;   // ... what the last tpc_track_sectors queued
    bool queueOutput = true;                // tpc_set_output_prefetch
    int64_t nRefetch = 0;
    // Phase II merging
    float sectorDphi = 0.f;
    MergePtrs mp{};
    bool merged = false, mergeFetched = false;
    cudaEvent_t evM0 = nullptr, evM1 = nullptr;
    int32_t* outNext = nullptr; int32_t* outPrev = nullptr; float* outMChi2 = nullptr; tpc_merged_track* outMerged = nullptr;
    int32_t* outSegments = nullptr; uint32_t* outMCount = nullptr; int64_t outMergeCap = 0;
    float mergeUs = 0.f; int32_t nMerged = 0, nMergeLinks = 0;
    // Phase II final fit
    tpc_refit_track* devRefit = nullptr;
    bool refitted = false, refitFetched = false;
    cudaEvent_t evR0 = nullptr, evR1 = nullptr;
    tpc_refit_track* outRefit = nullptr; int64_t outRefitCap = 0;
    float refitUs = 0.f;                   // how often the estimate was short (tpc_stats)
    RowGrid* hostGrid = nullptr;            // pinned
    RowMeta* hostMeta = nullptr;            // pinned
    uint32_t* hostSectorBase = nullptr;     // pinned
    uint32_t* hostCounters = nullptr;       // pinned
    uint32_t* hostRowStartBase = nullptr;   // pinned
    int maxBinsLaunch = 1;
    int maxRowN = 0;                        // clusters in the fullest (sector,row) of the loaded event
    bool k2Stage = false;                   // tpc_set_neighbour_staging

    std::vector<tpc_track> slTracks;        // tpc_track_event_sliced: the slices' results, concatenated
    std::vector<uint32_t> slIds;
    // results (pinned)
    tpc_track* outTracks = nullptr; int64_t outTracksCap = 0;
    uint32_t* outIds = nullptr; int64_t outIdsCap = 0;
    uint32_t counters[kNCounters] = {0};
    cudaEvent_t ev[8] = {nullptr};
    bool haveEvents = false;
    float kernelUs[8] = {0};
    int k5Blocks = 0, k6Blocks = 0, k6aBlocks = 0;
    size_t k5GridSmem = 0; bool k5SmemGrid = false;
};

namespace {

#define CUDA_TRY(t, expr)                                             \
    do {                                                              \
        cudaError_t _e = (expr);                                      \
        if (_e != cudaSuccess) { (t)->lastCuda = (int)_e; return TPC_E_CUDA; } \
    } while (0)

Layout make_layout(const tpc_tracker* t, int64_t maxClusters) {
    Layout L{};
    const int64_t NR = t->nRowsTotal;
    L.hitCap = maxClusters + (int64_t)kRowPad * NR + 16;
    L.binCap = (int64_t)((double)maxClusters * (double)t->P.grid_bins_per_hit) + 2 * NR + 16;
    L.maxTracklets = (int64_t)((double)maxClusters * (double)t->P.max_tracklets_per_cluster) + 4096;
    size_t o = 0;
    L.nGuards = 0;
    // every buffer is followed by a 256-byte guard zone (filled with a pattern by tpc_set_workspace, checked by
    // tpc_debug_check_guards: compute-sanitizer is not available on the target pool)
    auto take = [&](size_t bytes) {
        size_t r = o;
        o = align_up(o + bytes);
        if (L.nGuards < Layout::kMaxGuards) L.guard[L.nGuards++] = o;
        o += kAlign;
        return r;
    };
    L.inY = take(sizeof(float) * (maxClusters + 16));
    L.inZ = take(sizeof(float) * (maxClusters + 16));
    L.grid = take(sizeof(RowGrid) * (NR + 2));
    L.meta = take(sizeof(RowMeta) * (NR + 2));
    L.rowX = take(sizeof(float) * (t->nRows + 1));
    L.hits = take(sizeof(float2) * L.hitCap);
    L.orig = take(sizeof(uint32_t) * L.hitCap);
    L.binStart = take(sizeof(uint32_t) * L.binCap);
    L.buckets = take(sizeof(Bucket) * L.binCap);
    L.linkUp = take(sizeof(int32_t) * L.hitCap);
    L.linkDn = take(sizeof(int32_t) * L.hitCap);
    L.linkUpC = take(sizeof(int32_t) * L.hitCap);
    L.linkDnC = take(sizeof(int32_t) * L.hitCap);
    L.weight = take(sizeof(uint32_t) * L.hitCap);
    L.starts = take(sizeof(int4) * (maxClusters + 16));      // filed by pad row: a row's segment holds as many records as the row has clusters
    L.startsRaw = take(sizeof(int4) * L.maxTracklets);
    L.rowHist = take(sizeof(uint32_t) * (kMaxRows + 1));
    L.rowStartBase = take(sizeof(uint32_t) * (kMaxRows + 2));
    L.recs = take(sizeof(TrackletRec) * L.maxTracklets);
    L.rowHit = take(sizeof(int32_t) * L.maxTracklets * t->rhStride);
    L.tracks = take(sizeof(tpc_track) * L.maxTracklets);
    L.clusterIds = take(sizeof(uint32_t) * (maxClusters + 16));
    L.clusterPos = take(sizeof(uint32_t) * (maxClusters + 16));
    L.clusterRow = take(sizeof(uint8_t) * (maxClusters + 16));
    L.refit = take(sizeof(tpc_refit_track) * L.maxTracklets);
    L.counters = take(sizeof(uint32_t) * (kNCounters + kMaxPending));
    L.sectorGidBase = take(sizeof(uint32_t) * (t->nSec + 1));
    // K7 (Phase II merging): per-track words, sized like the track output
    const int64_t TC = L.maxTracklets;
    L.mKey = take(4 * TC); L.mOrder = take(4 * TC); L.mBestIn = take(8 * TC); L.mOut = take(4 * TC); L.mOutChi2 = take(4 * TC);
    L.mNext = take(4 * TC); L.mPrev = take(4 * TC); L.mChi2 = take(4 * TC); L.mMerged = take(sizeof(tpc_merged_track) * TC);
    L.mSegments = take(4 * TC); L.mBinStart = take(4 * (NR + 4)); L.mBinCursor = take(4 * (NR + 4)); L.mCount = take(16);
    L.total = o;
    return L;
}

// Launch `kernel` on stream s, as the programmatic dependent of the kernel before it if pdl (the kernel then starts
// when that one has triggered or finished, and waits for its completion itself: grid_dep_wait in device_types.cuh).
template <class... KArgs, class... Args>
cudaError_t launch_dep(bool pdl, void (*kernel)(KArgs...), int grid, int block, size_t smem, cudaStream_t s, Args... args) {
    cudaLaunchConfig_t cfg{};
    cfg.gridDim = dim3((unsigned)grid); cfg.blockDim = dim3((unsigned)block); cfg.dynamicSmemBytes = smem; cfg.stream = s;
    cudaLaunchAttribute attr[1];
    attr[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
    attr[0].val.programmaticStreamSerializationAllowed = 1;
    cfg.attrs = attr; cfg.numAttrs = pdl ? 1 : 0;
    return cudaLaunchKernelEx(&cfg, kernel, KArgs(args)...);
}

void bind_pointers(tpc_tracker* t) {
    char* w = t->ws;
    const Layout& L = t->L;
    DevPtrs& d = t->dev;
    d.inY = (const float*)(w + L.inY); d.inZ = (const float*)(w + L.inZ);
    d.grid = (RowGrid*)(w + L.grid); d.meta = (const RowMeta*)(w + L.meta); d.rowX = (const float*)(w + L.rowX);
    d.hits = (float2*)(w + L.hits); d.orig = (uint32_t*)(w + L.orig); d.binStart = (uint32_t*)(w + L.binStart); d.buckets = (Bucket*)(w + L.buckets);
    d.linkUp = (int32_t*)(w + L.linkUp); d.linkDn = (int32_t*)(w + L.linkDn);
    d.linkUpC = (int32_t*)(w + L.linkUpC); d.linkDnC = (int32_t*)(w + L.linkDnC);
    d.weight = (uint32_t*)(w + L.weight); d.starts = (int4*)(w + L.starts); d.startsRaw = (int4*)(w + L.startsRaw); d.rowHist = (uint32_t*)(w + L.rowHist); d.rowStartBase = (const uint32_t*)(w + L.rowStartBase);
    d.recs = (TrackletRec*)(w + L.recs); d.rowHit = (int32_t*)(w + L.rowHit);
    d.tracks = (tpc_track*)(w + L.tracks); d.clusterIds = (uint32_t*)(w + L.clusterIds);
    d.clusterPos = (uint32_t*)(w + L.clusterPos); d.clusterRow = (uint8_t*)(w + L.clusterRow);
    d.counters = (uint32_t*)(w + L.counters); d.sectorGidBase = (uint32_t*)(w + L.sectorGidBase);
    d.nRowsTotal = t->nRowsTotal; d.maxTracklets = (int32_t)std::min<int64_t>(L.maxTracklets, 0x7fffffff);
    d.rhStride = t->rhStride;
    MergePtrs& m = t->mp;
    m.tracks = d.tracks; m.clusterIds = d.clusterIds; m.counters = d.counters;
    m.key = (uint32_t*)(w + L.mKey); m.binStart = (uint32_t*)(w + L.mBinStart); m.binCursor = (uint32_t*)(w + L.mBinCursor);
    m.order = (uint32_t*)(w + L.mOrder); m.bestIn = (unsigned long long*)(w + L.mBestIn); m.out = (int32_t*)(w + L.mOut);
    m.outChi2 = (float*)(w + L.mOutChi2); m.next = (int32_t*)(w + L.mNext); m.prev = (int32_t*)(w + L.mPrev);
    m.chi2 = (float*)(w + L.mChi2); m.merged = (tpc_merged_track*)(w + L.mMerged); m.segments = (int32_t*)(w + L.mSegments);
    m.mcount = (uint32_t*)(w + L.mCount); m.nBins = t->nRowsTotal;
    t->devRefit = (tpc_refit_track*)(w + L.refit);
}

// Page-locked host memory (cudaMallocHost / cudaHostRegister, e.g. a pinned torch tensor): the DMA engine can read it
// directly, so large loads skip the copy into the library's own pinned mirror.
bool is_pinned_host_pointer(const void* p) {
    cudaPointerAttributes a;
    if (cudaPointerGetAttributes(&a, p) != cudaSuccess) { cudaGetLastError(); return false; }
    return a.type == cudaMemoryTypeHost;
}

bool is_device_pointer(const void* p) {
    cudaPointerAttributes a;
    if (cudaPointerGetAttributes(&a, p) != cudaSuccess) { cudaGetLastError(); return false; }
    return a.type == cudaMemoryTypeDevice || a.type == cudaMemoryTypeManaged;
}

int ensure_host_stage(tpc_tracker* t, int64_t need) {
    if (need <= t->hostCap) return TPC_OK;
    int64_t cap = std::max<int64_t>(need, t->hostCap * 2);
    cap = std::min<int64_t>(std::max<int64_t>(cap, 1 << 16), std::max<int64_t>(t->maxClusters, need));
    float *ny = nullptr, *nz = nullptr;
    CUDA_TRY(t, cudaMallocHost(&ny, sizeof(float) * cap));
    CUDA_TRY(t, cudaMallocHost(&nz, sizeof(float) * cap));
    if (t->hostY) {
        // pending async uploads read the old buffers: drain them first
        CUDA_TRY(t, cudaStreamSynchronize(t->stream));
        std::memcpy(ny, t->hostY, sizeof(float) * t->hostCap);
        std::memcpy(nz, t->hostZ, sizeof(float) * t->hostCap);
        cudaFreeHost(t->hostY); cudaFreeHost(t->hostZ);
    }
    t->hostY = ny; t->hostZ = nz; t->hostCap = cap;
    return TPC_OK;
}

// Upload the pending host-staged range [dirtyLo, dirtyHi) (one copy per array).
int flush_dirty(tpc_tracker* t) {
    if (t->dirtyHi <= t->dirtyLo) return TPC_OK;
    const int64_t lo = t->dirtyLo, cnt = t->dirtyHi - t->dirtyLo;
    CUDA_TRY(t, cudaMemcpyAsync((float*)t->dev.inY + lo, t->hostY + lo, sizeof(float) * cnt, cudaMemcpyHostToDevice, t->stream));
    CUDA_TRY(t, cudaMemcpyAsync((float*)t->dev.inZ + lo, t->hostZ + lo, sizeof(float) * cnt, cudaMemcpyHostToDevice, t->stream));
    if (!t->evUpload) CUDA_TRY(t, cudaEventCreateWithFlags(&t->evUpload, cudaEventDisableTiming));
    CUDA_TRY(t, cudaEventRecord(t->evUpload, t->stream));
    t->uploadPending = true;
    t->dirtyLo = t->dirtyHi = 0;
    return TPC_OK;
}

// Host "initialisation" of an event (PAPER.md:66 host pre-processing, reduced to a prefix sum over row counts):
// canonical id bases, padded row offsets, bin capacities; uploads the row table and any host-staged clusters.
int finalize_event(tpc_tracker* t) {
    if (t->finalized) return TPC_OK;
    const int NR = t->nRowsTotal;
    if (!t->hostGrid) {
        CUDA_TRY(t, cudaMallocHost(&t->hostGrid, sizeof(RowGrid) * (NR + 2)));
        CUDA_TRY(t, cudaMallocHost(&t->hostMeta, sizeof(RowMeta) * (NR + 2)));
        CUDA_TRY(t, cudaMallocHost(&t->hostSectorBase, sizeof(uint32_t) * (t->nSec + 1)));
        CUDA_TRY(t, cudaMallocHost(&t->hostCounters, sizeof(uint32_t) * kNCounters));
        CUDA_TRY(t, cudaMallocHost(&t->hostRowStartBase, sizeof(uint32_t) * (kMaxRows + 2)));
        CUDA_TRY(t, cudaEventCreateWithFlags(&t->evTables, cudaEventDisableTiming));
    } else if (t->tablesPending) {
        CUDA_TRY(t, cudaEventSynchronize(t->evTables));  // the previous upload may still read the host tables (the
        t->tablesPending = false;                        // kernels behind it are not waited for)
    }
    int64_t gid = 0, hitOff = 0, binOff = 0;
    int maxBins = 1, maxRow = 0;
    for (int i = 0; i < NR; i++) {
        RowGrid& G = t->hostGrid[i];
        RowMeta& M = t->hostMeta[i];
        if (i % t->nRows == 0) t->hostSectorBase[i / t->nRows] = (uint32_t)gid;
        const int n = t->rowN[i];
        G.hitOff = (int32_t)hitOff; G.binOff = (int32_t)binOff;
        G.nY = G.nZ = 1; G.y0 = G.z0 = 0.f; G.invY = G.invZ = 1.f;
        M.n = n; M.inOff = t->rowIn[i]; M.gidBase = (uint32_t)gid;
        M.maxBins = (int)std::max<int64_t>(1, std::min<int64_t>((int64_t)((double)n * (double)t->P.grid_bins_per_hit), kMaxBinsPerRow));
        maxBins = std::max(maxBins, M.maxBins);
        maxRow = std::max(maxRow, n);
        gid += n;
        hitOff += (n + kRowPad - 1) / kRowPad * kRowPad;
        binOff += M.maxBins + 1;
    }
    t->hostSectorBase[t->nSec] = (uint32_t)gid;
    {   // where each pad row's segment of the by-row start list begins: prefix over rows of the clusters per row
        uint64_t run = 0;
        for (int r = 0; r <= t->nRows; r++) {
            t->hostRowStartBase[r] = (uint32_t)run;
            if (r < t->nRows) for (int sct = 0; sct < t->nSec; sct++) run += (uint64_t)t->rowN[sct * t->nRows + r];
        }
    }
    for (int s = 0; s < t->nSec; s++)
        if ((int64_t)t->hostSectorBase[s + 1] - (int64_t)t->hostSectorBase[s] > 0x00FFFFFF) return TPC_E_ARG;  // key field
    t->nClusters = gid;
    t->maxBinsLaunch = maxBins;
    t->maxRowN = maxRow;
    if (gid > t->maxClusters || hitOff > t->L.hitCap || binOff > t->L.binCap) return TPC_E_NOMEM;
    CUDA_TRY(t, cudaMemcpyAsync(t->dev.grid, t->hostGrid, sizeof(RowGrid) * NR, cudaMemcpyHostToDevice, t->stream));
    CUDA_TRY(t, cudaMemcpyAsync((void*)t->dev.meta, t->hostMeta, sizeof(RowMeta) * NR, cudaMemcpyHostToDevice, t->stream));
    CUDA_TRY(t, cudaMemcpyAsync(t->dev.sectorGidBase, t->hostSectorBase, sizeof(uint32_t) * (t->nSec + 1),
                                cudaMemcpyHostToDevice, t->stream));
    CUDA_TRY(t, cudaMemcpyAsync((void*)t->dev.rowStartBase, t->hostRowStartBase, sizeof(uint32_t) * (t->nRows + 1),
                                cudaMemcpyHostToDevice, t->stream));
    CUDA_TRY(t, cudaEventRecord(t->evTables, t->stream));
    t->tablesPending = true;
    {
        int rc = flush_dirty(t);
        if (rc != TPC_OK) return rc;
    }
    t->finalized = true;
    return TPC_OK;
}

int stage_clusters(tpc_tracker* t, int64_t at, int64_t n, const float* y, const float* z) {
    if (n == 0) return TPC_OK;
    if (is_device_pointer(y)) {
        if (t->dirtyHi > t->dirtyLo && at < t->dirtyHi && at + n > t->dirtyLo) {   // a row replaced in place: the pending
            int rc = flush_dirty(t);                                              // host range must not overwrite it later
            if (rc != TPC_OK) return rc;
        }
        CUDA_TRY(t, cudaMemcpyAsync((float*)t->dev.inY + at, y, sizeof(float) * n, cudaMemcpyDeviceToDevice, t->stream));
        CUDA_TRY(t, cudaMemcpyAsync((float*)t->dev.inZ + at, z, sizeof(float) * n, cudaMemcpyDeviceToDevice, t->stream));
    } else if (n >= (1 << 16) && is_pinned_host_pointer(y) && is_pinned_host_pointer(z)) {
        // large page-locked buffers: DMA straight from the caller's memory.  The call returns when the copy is QUEUED
        // (DMA || kernels): the caller must not touch the buffers before tpc_wait_input (tpctrk.h)
        int rc = flush_dirty(t);     // keep the order of uploads
        if (rc != TPC_OK) return rc;
        CUDA_TRY(t, cudaMemcpyAsync((float*)t->dev.inY + at, y, sizeof(float) * n, cudaMemcpyHostToDevice, t->stream));
        CUDA_TRY(t, cudaMemcpyAsync((float*)t->dev.inZ + at, z, sizeof(float) * n, cudaMemcpyHostToDevice, t->stream));
        if (!t->evUpload) CUDA_TRY(t, cudaEventCreateWithFlags(&t->evUpload, cudaEventDisableTiming));
        CUDA_TRY(t, cudaEventRecord(t->evUpload, t->stream));
        t->uploadPending = true;
    } else {
        int rc = ensure_host_stage(t, at + n);
        if (rc != TPC_OK) return rc;
        if (t->uploadPending) {   // an earlier upload may still read the pinned mirror
            CUDA_TRY(t, cudaEventSynchronize(t->evUpload));
            t->uploadPending = false;
        }
        if (t->dirtyHi > t->dirtyLo && at != t->dirtyHi) {   // not contiguous with the pending range (e.g. device
            rc = flush_dirty(t);                              // loads in between): upload what we have first
            if (rc != TPC_OK) return rc;
            CUDA_TRY(t, cudaEventSynchronize(t->evUpload));
            t->uploadPending = false;
        }
        std::memcpy(t->hostY + at, y, sizeof(float) * n);
        std::memcpy(t->hostZ + at, z, sizeof(float) * n);
        if (t->dirtyHi == t->dirtyLo) { t->dirtyLo = at; t->dirtyHi = at + n; }
        else t->dirtyHi = at + n;
    }
    return TPC_OK;
}

int ensure_out(tpc_tracker* t, int64_t nT, int64_t nC) {
    if (nT > t->outTracksCap) {
        tpc_track* nb = nullptr;
        const int64_t cap = std::max<int64_t>(nT, 1024) * 3 / 2;
        CUDA_TRY(t, cudaMallocHost(&nb, sizeof(tpc_track) * cap));
        if (t->outTracks) { CUDA_TRY(t, cudaStreamSynchronize(t->stream)); std::memcpy(nb, t->outTracks, sizeof(tpc_track) * t->outTracksCap); cudaFreeHost(t->outTracks); }
        t->outTracks = nb; t->outTracksCap = cap;
    }
    if (nC > t->outIdsCap) {
        uint32_t* nb = nullptr;
        const int64_t cap = std::max<int64_t>(nC, 1024) * 3 / 2;
        CUDA_TRY(t, cudaMallocHost(&nb, sizeof(uint32_t) * cap));
        if (t->outIds) { CUDA_TRY(t, cudaStreamSynchronize(t->stream)); std::memcpy(nb, t->outIds, sizeof(uint32_t) * t->outIdsCap); cudaFreeHost(t->outIds); }
        t->outIds = nb; t->outIdsCap = cap;
    }
    return TPC_OK;
}

// Queue, behind K6, the download of the counters and of the estimated prefix of the result.
int queue_download(tpc_tracker* t) {
    cudaStream_t s = t->stream;
    if (!t->evDone) CUDA_TRY(t, cudaEventCreateWithFlags(&t->evDone, cudaEventDisableTiming));
    CUDA_TRY(t, cudaMemcpyAsync(t->hostCounters, t->dev.counters, sizeof(uint32_t) * kNCounters, cudaMemcpyDeviceToHost, s));
    t->queuedTracks = t->queuedIds = 0;
    if (t->queueOutput && t->nClusters > 0) {
        // first event: one track per 64 clusters, every cluster in a track; later: the last event's counts + 25 %
        int64_t eT = t->estTracks > 0 ? t->estTracks : t->nClusters / 64 + 256;
        int64_t eC = t->estIds > 0 ? t->estIds : t->nClusters;
        eT = std::min<int64_t>(eT, t->dev.maxTracklets);
        eC = std::min<int64_t>(eC, t->nClusters);
        int rc = ensure_out(t, eT, eC);
        if (rc != TPC_OK) return rc;
        CUDA_TRY(t, cudaMemcpyAsync(t->outTracks, t->dev.tracks, sizeof(tpc_track) * eT, cudaMemcpyDeviceToHost, s));
        CUDA_TRY(t, cudaMemcpyAsync(t->outIds, t->dev.clusterIds, sizeof(uint32_t) * eC, cudaMemcpyDeviceToHost, s));
        t->queuedTracks = eT; t->queuedIds = eC;
    }
    CUDA_TRY(t, cudaEventRecord(t->evDone, s));
    return TPC_OK;
}

// ---- debug-dump conversion kernels (tests only; not on the hot path)
__global__ void dump_links_kernel(DevPtrs d, int nRows, int64_t N, int32_t* out) {
    const int rowId = blockIdx.x, r = rowId % nRows;
    const RowGrid R = d.grid[rowId];
    const RowMeta M = d.meta[rowId];
    for (int k = threadIdx.x; k < M.n; k += blockDim.x) {
        const int64_t g = (int64_t)d.orig[R.hitOff + k];
        const int32_t* src[4] = {d.linkUp, d.linkDn, d.linkUpC, d.linkDnC};
        for (int w = 0; w < 4; w++) {
            const int l = src[w][R.hitOff + k];
            int v = -1;
            if (l >= 0) {
                const bool upw = (w % 2) == 0;
                if ((upw && r + 1 < nRows) || (!upw && r >= 1)) {
                    const int nb = rowId + (upw ? 1 : -1);
                    v = (int)(d.orig[d.grid[nb].hitOff + l] - d.meta[nb].gidBase);
                }
            }
            out[(int64_t)w * N + g] = v;
        }
    }
}
__global__ void dump_starts_kernel(DevPtrs d, unsigned n, uint32_t* out) {
    const unsigned i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n) return;
    const int4 s = d.startsRaw[i];      // append order (the row-ordered copy exists only for the phased K5 kernel)
    out[i] = d.orig[d.grid[s.x].hitOff + s.y];
}
__global__ void dump_rowhit_kernel(DevPtrs d, int nRows, unsigned n, int32_t* out) {
    const unsigned slot = blockIdx.x;
    if (slot >= n) return;
    const TrackletRec t = d.recs[slot];
    for (int r = threadIdx.x; r < nRows; r += blockDim.x) {
        int v = -1;
        if (r >= t.firstRow && r <= t.lastRow) {
            const int h = d.rowHit[(size_t)slot * d.rhStride + r];
            if (h >= 0) v = (int)(d.orig[h] - d.meta[t.sector * nRows + r].gidBase);
        }
        out[(size_t)slot * nRows + r] = v;
    }
}
__global__ void dump_owner_kernel(DevPtrs d, int nRows, uint32_t* out) {
    const int rowId = blockIdx.x;
    const RowGrid R = d.grid[rowId];
    const RowMeta M = d.meta[rowId];
    const uint32_t sb = d.sectorGidBase[rowId / nRows];
    for (int k = threadIdx.x; k < M.n; k += blockDim.x) {
        const uint32_t w = d.weight[R.hitOff + k];
        out[d.orig[R.hitOff + k]] = w ? sb + (0x00FFFFFFu - (w & 0x00FFFFFFu)) : 0xFFFFFFFFu;
    }
}

}  // namespace

extern "C" {

void tpc_default_params(tpc_params* p) {
    if (!p) return;
    p->err2_y = 0.01f; p->err2_z = 0.01f;
    p->nf_ty = 1.0f; p->nf_tz = 1.5f; p->nf_c = 0.5f; p->nf_d2max = 0.25f;
    p->kf_css0 = 1.0f; p->kf_ctt0 = 10.0f; p->kf_ckk0 = 100.0f; p->kf_smax = 0.95f;
    p->road_nsig = 4.0f; p->road_max = 2.0f;
    p->max_gap = 4; p->min_hits = 10; p->seed_min_chain = 3;
    p->merge_chi2 = 50.0f; p->merge_max_row_gap = 40;
    p->field_ar = 0.0f; p->field_az = 0.0f; p->ms_x0_inv = 0.0f;
    p->max_tracklets_per_cluster = 0.1f;
    p->grid_bins_per_hit = 2.0f;
}

int tpc_tracker_create(const tpc_geometry* g, float bz_tesla, tpc_tracker** out) {
    if (!g || !out || !g->row_x) return TPC_E_ARG;
    if (g->n_sectors < 1 || g->n_rows < 3 || g->n_rows > kMaxRows) return TPC_E_ARG;
    if ((int64_t)g->n_sectors * g->n_rows > (1 << 24)) return TPC_E_ARG;
    for (int i = 1; i < g->n_rows; i++)
        if (!(g->row_x[i] > g->row_x[i - 1])) return TPC_E_ARG;
    tpc_tracker* t = new (std::nothrow) tpc_tracker();
    if (!t) return TPC_E_NOMEM;
    t->nSec = g->n_sectors; t->nRows = g->n_rows; t->nRowsTotal = g->n_sectors * g->n_rows;
    t->rhStride = (g->n_rows + 31) / 32 * 32;
    t->rowX.assign(g->row_x, g->row_x + g->n_rows);
    if (g->params) t->P = *g->params; else tpc_default_params(&t->P);
    {
        // the kernels' branch-free reciprocals and square roots assume positive finite variances and roads
        // (kernels_kf.cuh rcp_rn_inrange / sqrt_rn_inrange): everything else is refused here
        const tpc_params& P = t->P;
        auto pos = [](float v) { return v > 0.f && v < 1e30f; };              // false for NaN, inf, <= 0
        auto nonneg = [](float v) { return v >= 0.f && v < 1e30f; };
        const bool ok = pos(P.err2_y) && pos(P.err2_z) && pos(P.kf_css0) && pos(P.kf_ctt0) && pos(P.kf_ckk0) &&
                        pos(P.road_nsig) && pos(P.road_max) && P.kf_smax > 0.f && P.kf_smax < 1.f &&
                        nonneg(P.nf_ty) && nonneg(P.nf_tz) && nonneg(P.nf_c) && nonneg(P.nf_d2max) &&
                        P.seed_min_chain >= 2 && P.min_hits >= 1 && P.max_gap >= 0 && pos(P.max_tracklets_per_cluster) &&
                        P.grid_bins_per_hit >= 0.25f && P.grid_bins_per_hit <= 64.f && nonneg(P.merge_chi2) && P.merge_max_row_gap >= 0 &&
                        nonneg(P.ms_x0_inv) && std::abs(P.field_ar) < 1e30f && std::abs(P.field_az) < 1e30f && bz_tesla == bz_tesla && std::abs(bz_tesla) < 1e3f;
        if (!ok) { delete t; return TPC_E_ARG; }
    }
    t->sectorDphi = g->sector_dphi;
    t->bz = bz_tesla;
    t->CB = (float)(-0.299792458e-2 * (double)bz_tesla);   // kappa = (q/pT) * CB, constant field
    t->rowN.assign(t->nRowsTotal, 0); t->rowIn.assign(t->nRowsTotal, 0); t->rowCap.assign(t->nRowsTotal, 0);
    *out = t;
    return TPC_OK;
}

void tpc_tracker_destroy(tpc_tracker* t) {
    if (!t) return;
    if (t->stream || t->ws) cudaStreamSynchronize(t->stream);
    if (t->hostY) cudaFreeHost(t->hostY);
    if (t->hostZ) cudaFreeHost(t->hostZ);
    if (t->hostGrid) cudaFreeHost(t->hostGrid);
    if (t->hostMeta) cudaFreeHost(t->hostMeta);
    if (t->hostSectorBase) cudaFreeHost(t->hostSectorBase);
    if (t->hostCounters) cudaFreeHost(t->hostCounters);
    if (t->hostRowStartBase) cudaFreeHost(t->hostRowStartBase);
    if (t->outTracks) cudaFreeHost(t->outTracks);
    if (t->outIds) cudaFreeHost(t->outIds);
    if (t->haveEvents) for (auto& e : t->ev) cudaEventDestroy(e);
    if (t->evUpload) cudaEventDestroy(t->evUpload);
    if (t->evTables) cudaEventDestroy(t->evTables);
    if (t->evDone) cudaEventDestroy(t->evDone);
    if (t->evM0) cudaEventDestroy(t->evM0);
    if (t->evM1) cudaEventDestroy(t->evM1);
    if (t->evR0) cudaEventDestroy(t->evR0);
    if (t->evR1) cudaEventDestroy(t->evR1);
    if (t->outRefit) cudaFreeHost(t->outRefit);
    for (void* q : {(void*)t->outNext, (void*)t->outPrev, (void*)t->outMChi2, (void*)t->outMerged, (void*)t->outSegments, (void*)t->outMCount})
        if (q) cudaFreeHost(q);
    delete t;
}

int tpc_set_kernel_timing(tpc_tracker* t, int on) {
    if (!t) return TPC_E_ARG;
    t->kernelTiming = on != 0;
    return TPC_OK;
}

int tpc_set_dependent_launch(tpc_tracker* t, int on) {
    if (!t) return TPC_E_ARG;
    t->dependentLaunch = on != 0;
    return TPC_OK;
}

int tpc_set_neighbour_staging(tpc_tracker* t, int on) {
    if (!t) return TPC_E_ARG;
    t->k2Stage = on != 0;
    return TPC_OK;
}

int tpc_set_output_prefetch(tpc_tracker* t, int on) {
    if (!t) return TPC_E_ARG;
    t->queueOutput = on != 0;
    return TPC_OK;
}

int tpc_wait_input(tpc_tracker* t) {
    if (!t) return TPC_E_ARG;
    if (t->uploadPending) { CUDA_TRY(t, cudaEventSynchronize(t->evUpload)); t->uploadPending = false; }
    if (t->tablesPending) { CUDA_TRY(t, cudaEventSynchronize(t->evTables)); t->tablesPending = false; }
    return TPC_OK;
}

int tpc_set_stream(tpc_tracker* t, void* cuda_stream) {
    if (!t) return TPC_E_ARG;
    t->stream = (cudaStream_t)cuda_stream;
    return TPC_OK;
}

size_t tpc_workspace_bytes(const tpc_tracker* t, int64_t max_clusters) {
    if (!t || max_clusters < 0) return 0;
    return make_layout(t, max_clusters).total;
}

int tpc_set_workspace(tpc_tracker* t, void* dev_ptr, size_t bytes) {
    if (!t || !dev_ptr || ((uintptr_t)dev_ptr % kAlign) != 0) return TPC_E_ARG;
    // capacity = largest max_clusters whose layout fits (the layout is monotone in max_clusters)
    if (make_layout(t, 0).total > bytes) return TPC_E_NOMEM;
    int64_t lo = 0, hi = 1;
    while (make_layout(t, hi).total <= bytes && hi < (int64_t)1 << 31) hi *= 2;
    while (hi - lo > 1) {
        const int64_t mid = lo + (hi - lo) / 2;
        if (make_layout(t, mid).total <= bytes) lo = mid; else hi = mid;
    }
    lo = std::min<int64_t>(lo, ((int64_t)1 << 31) - 65536);
    t->ws = (char*)dev_ptr; t->wsBytes = bytes; t->maxClusters = lo;
    t->L = make_layout(t, lo);
    bind_pointers(t);
    for (int g = 0; g < t->L.nGuards; g++)
        CUDA_TRY(t, cudaMemsetAsync(t->ws + t->L.guard[g], 0xA5, kAlign, t->stream));
    CUDA_TRY(t, cudaMemcpyAsync((void*)t->dev.rowX, t->rowX.data(), sizeof(float) * t->nRows, cudaMemcpyHostToDevice, t->stream));
    CUDA_TRY(t, cudaStreamSynchronize(t->stream));
    if (!t->haveEvents) {
        for (auto& e : t->ev) CUDA_TRY(t, cudaEventCreate(&e));
        t->haveEvents = true;
        int dev = 0, sms = 0, occ5 = 0, occ6 = 0;
        CUDA_TRY(t, cudaGetDevice(&dev));
        CUDA_TRY(t, cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev));
        // K5 keeps the whole row table in shared memory when it fits (one block per SM)
        t->k5GridSmem = sizeof(RowGrid) * (size_t)t->nRowsTotal;
        {
            // dynamic + static shared memory of BOTH instantiations must fit the opt-in limit; otherwise (or if the
            // attribute cannot be set) the same kernels read the table from global memory
            int optin = 0;
            CUDA_TRY(t, cudaDeviceGetAttribute(&optin, cudaDevAttrMaxSharedMemoryPerBlockOptin, dev));
            cudaFuncAttributes fa{}, fb{};
            CUDA_TRY(t, cudaFuncGetAttributes(&fa, k5_construct_free<true>));
            CUDA_TRY(t, cudaFuncGetAttributes(&fb, k5_construct_phased<true>));
            const size_t stat = std::max(fa.sharedSizeBytes, fb.sharedSizeBytes);
            t->k5SmemGrid = t->k5GridSmem + stat <= (size_t)optin;
            if (t->k5SmemGrid) {
                cudaError_t e1 = cudaFuncSetAttribute(k5_construct_free<true>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)t->k5GridSmem);
                cudaError_t e2 = cudaFuncSetAttribute(k5_construct_phased<true>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)t->k5GridSmem);
                if (e1 != cudaSuccess || e2 != cudaSuccess) { cudaGetLastError(); t->k5SmemGrid = false; }
            }
        }
        occ5 = 1;   // one persistent block per SM (both instantiations must see the same grid)
        CUDA_TRY(t, cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ6, k6_select, kK6Threads, 0));
        t->k5Blocks = sms * std::max(1, occ5);
        t->k6Blocks = sms * std::max(1, occ6);
        int occ6a = 0;
        CUDA_TRY(t, cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ6a, k6_weights, kK6Threads, 0));
        t->k6aBlocks = sms * std::max(1, occ6a);
    }
    return tpc_reset_event(t);
}

int tpc_reset_event(tpc_tracker* t) {
    if (!t) return TPC_E_ARG;
    std::fill(t->rowN.begin(), t->rowN.end(), 0);
    std::fill(t->rowIn.begin(), t->rowIn.end(), 0);
    std::fill(t->rowCap.begin(), t->rowCap.end(), 0);
    t->cursor = 0; t->nClusters = 0; t->dirtyLo = t->dirtyHi = 0;
    t->finalized = t->tracked = t->fetched = false;
    return TPC_OK;
}

int tpc_load_clusters(tpc_tracker* t, int sector, int row, int n, const float* x, const float* y, const float* z) {
    (void)x;   // R-13: the tracker uses the pad-row x
    if (!t || sector < 0 || sector >= t->nSec || row < 0 || row >= t->nRows || n < 0) return TPC_E_ARG;
    if (n > 0 && (!y || !z)) return TPC_E_ARG;
    if (!t->ws) return TPC_E_STATE;
    const int i = sector * t->nRows + row;
    // a (sector,row) that is loaded again keeps its staging slots if the new load fits the slots reserved for it, else
    // it is appended (the old slots stay unused until tpc_reset_event; tpctrk.h)
    const bool reuse = n <= t->rowCap[i];
    if (!reuse && t->cursor + n > t->maxClusters) return TPC_E_NOMEM;
    const int64_t at = reuse ? t->rowIn[i] : t->cursor;
    int rc = stage_clusters(t, at, n, y, z);
    if (rc != TPC_OK) return rc;
    t->rowN[i] = n; t->rowIn[i] = (int32_t)at;
    if (!reuse) { t->rowCap[i] = n; t->cursor += n; }
    t->finalized = t->tracked = t->fetched = false;
    return TPC_OK;
}

int tpc_load_event(tpc_tracker* t, const int32_t* row_counts, const float* y, const float* z) {
    if (!t || !row_counts) return TPC_E_ARG;
    if (!t->ws) return TPC_E_STATE;
    int64_t total = 0;
    for (int i = 0; i < t->nRowsTotal; i++) {
        if (row_counts[i] < 0) return TPC_E_ARG;
        total += row_counts[i];
    }
    if (total > 0 && (!y || !z)) return TPC_E_ARG;
    if (total > t->maxClusters) return TPC_E_NOMEM;
    tpc_reset_event(t);
    int64_t off = 0;
    for (int i = 0; i < t->nRowsTotal; i++) { t->rowN[i] = t->rowCap[i] = row_counts[i]; t->rowIn[i] = (int32_t)off; off += row_counts[i]; }
    t->cursor = total;
    int rc = stage_clusters(t, 0, total, y, z);
    if (rc != TPC_OK) return rc;
    return finalize_event(t);
}

int tpc_track_sectors(tpc_tracker* t) {
    if (!t) return TPC_E_ARG;
    if (!t->ws) return TPC_E_STATE;
    int rc = finalize_event(t);
    if (rc != TPC_OK) return rc;
    const DevPtrs d = t->dev;
    DevParams dp; dp.P = t->P; dp.CB = t->CB; dp.nSec = t->nSec; dp.nRows = t->nRows;
    const int NR = t->nRowsTotal;
    cudaStream_t s = t->stream;
    const bool timed = t->kernelTiming;     // events between the kernels only on request (tpctrk.h)
    t->timedCall = timed;
    CUDA_TRY(t, cudaEventRecord(t->ev[0], s));
    k1_sort_grid<<<NR, kK1Threads, sizeof(uint32_t) * (t->maxBinsLaunch + 1), s>>>(d);
    if (timed) CUDA_TRY(t, cudaEventRecord(t->ev[1], s));
    // K2..K6: without events between them each kernel is launched as the programmatic dependent of the one before
    // (its launch is set up while that one still runs; K5 also stages its row table meanwhile, device_types.cuh
    // grid_dep_wait); with events they are ordinary launches.
#ifndef TPC_PDL
#define TPC_PDL 1
#endif
    const bool pdl = TPC_PDL && !timed && t->dependentLaunch;
    const int k5Blocks = t->k5Blocks, phW = kK5PhasedThreads / 32;
    {   // K2: a block per chunk of kK2Chunk sorted hits of a (sector,row): grid.y = chunks of the fullest row
        cudaLaunchConfig_t cfg{};
        cfg.gridDim = dim3((unsigned)NR, (unsigned)std::max(1, (t->maxRowN + kK2Chunk - 1) / kK2Chunk));
        cfg.blockDim = dim3(kK2Threads); cfg.stream = s;
        cudaLaunchAttribute attr[1];
        attr[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
        attr[0].val.programmaticStreamSerializationAllowed = 1;
        cfg.attrs = attr; cfg.numAttrs = pdl ? 1 : 0;
        // dense rows (time frames; the same criterion as K3's start order below): more cached down-candidates per thread
        const bool dense = t->nClusters > (int64_t)1000 * NR;
        if (t->k2Stage) CUDA_TRY(t, cudaLaunchKernelEx(&cfg, k2_neighbours<true, kK2Cap>, d, dp));
        else if (dense) CUDA_TRY(t, cudaLaunchKernelEx(&cfg, k2_neighbours<false, kK2CapDense>, d, dp));
        else CUDA_TRY(t, cudaLaunchKernelEx(&cfg, k2_neighbours<false, kK2Cap>, d, dp));
    }
    if (timed) CUDA_TRY(t, cudaEventRecord(t->ev[2], s));
    CUDA_TRY(t, launch_dep(pdl, k3_clean_start, NR, kK3Threads, 0, s, d, dp, t->nClusters > (int64_t)1000 * NR ? 1 : 0));
    if (timed) CUDA_TRY(t, cudaEventRecord(t->ev[3], s));
    // K5: one persistent block per SM; the phased and the free-running instantiation decide on the device (from the
    // number of start hits) which of them does the event, the other returns at once
    if (t->k5SmemGrid) {
        CUDA_TRY(t, launch_dep(pdl, k5_construct_phased<true>, k5Blocks, kK5PhasedThreads, t->k5GridSmem, s, d, dp));
        CUDA_TRY(t, launch_dep(pdl, k5_construct_free<true>, k5Blocks, kK5Threads, t->k5GridSmem, s, d, dp, phW));
    } else {
        CUDA_TRY(t, launch_dep(pdl, k5_construct_phased<false>, k5Blocks, kK5PhasedThreads, 0, s, d, dp));
        CUDA_TRY(t, launch_dep(pdl, k5_construct_free<false>, k5Blocks, kK5Threads, 0, s, d, dp, phW));
    }
    if (timed) CUDA_TRY(t, cudaEventRecord(t->ev[4], s));
    CUDA_TRY(t, launch_dep(pdl, k6_weights, t->k6aBlocks, kK6Threads, 0, s, d, dp, k5Blocks));
    if (timed) CUDA_TRY(t, cudaEventRecord(t->ev[5], s));
    CUDA_TRY(t, launch_dep(pdl, k6_select, 2 * t->k6Blocks, kK6Threads, 0, s, d, dp));   // measured: 2 waves of warps beat 1 here (45 vs 50 us), not in K6a
    CUDA_TRY(t, cudaEventRecord(t->ev[6], s));
    CUDA_TRY(t, cudaGetLastError());
    // "the tracker can estimate a buffer that is large enough to store all tracks and queue the transfer
    // of this buffer immediately [...] if the estimation was too small, the tracker can still fetch the rest": the
    // counters and an estimated prefix of the tracks and cluster ids go to pinned host memory right behind K6, so that
    // tpc_get_tracks waits once and normally copies nothing.
    rc = queue_download(t);
    if (rc != TPC_OK) return rc;
    t->tracked = true; t->fetched = false; t->merged = false; t->mergeFetched = false; t->refitted = false; t->refitFetched = false;
    return TPC_OK;
}

int tpc_merge_tracks(tpc_tracker* t) {
    if (!t) return TPC_E_ARG;
    if (!t->tracked) return TPC_E_STATE;
    cudaStream_t s = t->stream;
    if (!t->evM0) { CUDA_TRY(t, cudaEventCreate(&t->evM0)); CUDA_TRY(t, cudaEventCreate(&t->evM1)); }
    DevParams dp; dp.P = t->P; dp.CB = t->CB; dp.nSec = t->nSec; dp.nRows = t->nRows;
    const MergePtrs m = t->mp;
    const int perSide = t->nSec >= 36 ? 18 : t->nSec;       // sectors per TPC side (tpctrk.h)
    const float cosB = (float)std::cos((double)t->sectorDphi), sinB = (float)std::sin((double)t->sectorDphi);
    const int grid = t->k6Blocks;                            // grid-stride over the tracks (their number is on the device)
    CUDA_TRY(t, cudaEventRecord(t->evM0, s));
    // the six kernels behind k7_init as programmatic dependents of the one before (each waits for it first thing:
    // what is saved is the launch gap, ~2 us each), unless the tracker shares the GPU (tpc_set_dependent_launch)
    const bool pdl = TPC_PDL && t->dependentLaunch;
    k7_init<<<grid, kK7Threads, 0, s>>>(m, t->nRows);
    CUDA_TRY(t, launch_dep(pdl, k7_hist, grid, kK7Threads, 0, s, m, t->nRows));
    CUDA_TRY(t, launch_dep(pdl, k7_scan, 1, 1024, 0, s, m));
    CUDA_TRY(t, launch_dep(pdl, k7_scatter, grid, kK7Threads, 0, s, m, t->nRows));
    CUDA_TRY(t, launch_dep(pdl, k7_match, grid, kK7Threads, 0, s, m, dp, perSide, cosB, sinB));
    CUDA_TRY(t, launch_dep(pdl, k7_link, grid, kK7Threads, 0, s, m));
    CUDA_TRY(t, launch_dep(pdl, k7_chains, grid, kK7Threads, 0, s, m));
    CUDA_TRY(t, cudaEventRecord(t->evM1, s));
    CUDA_TRY(t, cudaGetLastError());
    t->merged = true; t->mergeFetched = false; t->refitted = false; t->refitFetched = false;
    return TPC_OK;
}

int tpc_refit_tracks(tpc_tracker* t) {
    if (!t) return TPC_E_ARG;
    if (!t->merged) return TPC_E_STATE;
    cudaStream_t s = t->stream;
    if (!t->evR0) { CUDA_TRY(t, cudaEventCreate(&t->evR0)); CUDA_TRY(t, cudaEventCreate(&t->evR1)); }
    DevParams dp; dp.P = t->P; dp.CB = t->CB; dp.nSec = t->nSec; dp.nRows = t->nRows;
    const int perSide = t->nSec >= 36 ? 18 : t->nSec;
    const float cosB = (float)std::cos((double)t->sectorDphi), sinB = (float)std::sin((double)t->sectorDphi);
    CUDA_TRY(t, cudaEventRecord(t->evR0, s));
    k8_refit<<<t->k6Blocks, kK7Threads, 0, s>>>(t->mp, t->dev, dp, t->devRefit, perSide, cosB, sinB);
    CUDA_TRY(t, cudaEventRecord(t->evR1, s));
    CUDA_TRY(t, cudaGetLastError());
    t->refitted = true; t->refitFetched = false;
    return TPC_OK;
}

int tpc_get_refit(tpc_tracker* t, const tpc_refit_track** refit, int32_t* n_merged) {
    if (!t) return TPC_E_ARG;
    if (!t->refitted) return TPC_E_STATE;
    int rc = tpc_get_merged(t, nullptr, nullptr, nullptr, nullptr, nullptr, nullptr, nullptr);     // the counts
    if (rc != TPC_OK) return rc;
    const int64_t nM = t->nMerged;
    if (!t->refitFetched) {
        if (nM + 1 > t->outRefitCap) {
            if (t->outRefit) cudaFreeHost(t->outRefit);
            t->outRefitCap = std::max<int64_t>(nM + 1, 1024) * 3 / 2;
            CUDA_TRY(t, cudaMallocHost(&t->outRefit, sizeof(tpc_refit_track) * t->outRefitCap));
        }
        if (nM) CUDA_TRY(t, cudaMemcpyAsync(t->outRefit, t->devRefit, sizeof(tpc_refit_track) * nM, cudaMemcpyDeviceToHost, t->stream));
        CUDA_TRY(t, cudaStreamSynchronize(t->stream));
        float ms = 0.f;
        CUDA_TRY(t, cudaEventElapsedTime(&ms, t->evR0, t->evR1));
        t->refitUs = ms * 1000.f;
        t->refitFetched = true;
    }
    if (refit) *refit = t->outRefit;
    if (n_merged) *n_merged = (int32_t)nM;
    return TPC_OK;
}

int tpc_get_merged(tpc_tracker* t, const int32_t** next, const int32_t** prev, const float** chi2, int32_t* n_tracks,
                   const tpc_merged_track** merged, int32_t* n_merged, const int32_t** segments) {
    if (!t) return TPC_E_ARG;
    if (!t->merged) return TPC_E_STATE;
    int rc = tpc_sync(t);                     // the track counters (the merge kernels are behind them on the stream)
    if (rc != TPC_OK) return rc;
    const int64_t nT = t->counters[kNTracks];
    if (!t->mergeFetched) {
        if (nT + 1 > t->outMergeCap) {
            for (void* q : {(void*)t->outNext, (void*)t->outPrev, (void*)t->outMChi2, (void*)t->outMerged, (void*)t->outSegments})
                if (q) cudaFreeHost(q);
            const int64_t cap = std::max<int64_t>(nT + 1, 1024) * 3 / 2;
            CUDA_TRY(t, cudaMallocHost(&t->outNext, 4 * cap)); CUDA_TRY(t, cudaMallocHost(&t->outPrev, 4 * cap));
            CUDA_TRY(t, cudaMallocHost(&t->outMChi2, 4 * cap)); CUDA_TRY(t, cudaMallocHost(&t->outMerged, sizeof(tpc_merged_track) * cap));
            CUDA_TRY(t, cudaMallocHost(&t->outSegments, 4 * cap));
            if (!t->outMCount) CUDA_TRY(t, cudaMallocHost(&t->outMCount, 16));
            t->outMergeCap = cap;
        }
        cudaStream_t s = t->stream;
        const MergePtrs& m = t->mp;
        CUDA_TRY(t, cudaMemcpyAsync(t->outMCount, m.mcount, 8, cudaMemcpyDeviceToHost, s));
        if (nT) {
            CUDA_TRY(t, cudaMemcpyAsync(t->outNext, m.next, 4 * nT, cudaMemcpyDeviceToHost, s));
            CUDA_TRY(t, cudaMemcpyAsync(t->outPrev, m.prev, 4 * nT, cudaMemcpyDeviceToHost, s));
            CUDA_TRY(t, cudaMemcpyAsync(t->outMChi2, m.chi2, 4 * nT, cudaMemcpyDeviceToHost, s));
            CUDA_TRY(t, cudaMemcpyAsync(t->outMerged, m.merged, sizeof(tpc_merged_track) * nT, cudaMemcpyDeviceToHost, s));
            CUDA_TRY(t, cudaMemcpyAsync(t->outSegments, m.segments, 4 * nT, cudaMemcpyDeviceToHost, s));
        }
        CUDA_TRY(t, cudaStreamSynchronize(s));
        t->nMerged = (int32_t)t->outMCount[0];
        t->nMergeLinks = (int32_t)(nT - t->nMerged);
        float ms = 0.f;
        CUDA_TRY(t, cudaEventElapsedTime(&ms, t->evM0, t->evM1));
        t->mergeUs = ms * 1000.f;
        t->mergeFetched = true;
    }
    if (next) *next = t->outNext;
    if (prev) *prev = t->outPrev;
    if (chi2) *chi2 = t->outMChi2;
    if (n_tracks) *n_tracks = (int32_t)nT;
    if (merged) *merged = t->outMerged;
    if (n_merged) *n_merged = t->nMerged;
    if (segments) *segments = t->outSegments;
    return TPC_OK;
}

int tpc_launches_per_track(const tpc_tracker* t) { (void)t; return 7; }

int tpc_sync(tpc_tracker* t) {
    if (!t) return TPC_E_ARG;
    if (!t->tracked) return TPC_E_STATE;
    CUDA_TRY(t, cudaEventSynchronize(t->evDone));      // K1..K6, the counters and the queued part of the result
    t->uploadPending = false; t->tablesPending = false;    // (everything queued before it is complete as well)
    std::memcpy(t->counters, t->hostCounters, sizeof(t->counters));
    float total = 0.f;
    for (int i = 0; i < 6; i++) {
        float ms = 0.f;
        if (t->timedCall) CUDA_TRY(t, cudaEventElapsedTime(&ms, t->ev[i], t->ev[i + 1]));
        t->kernelUs[i] = ms * 1000.f;
    }
    CUDA_TRY(t, cudaEventElapsedTime(&total, t->ev[0], t->ev[6]));
    t->kernelUs[6] = total * 1000.f;
    // [7]: 1 if this event was the phased K5 kernel's, whose warps run the K6a weights pass themselves (same test as
    // k5_phased_mode on the device); K6a's own launch then only did the few groups the last warps left to it
    const unsigned nTotal = (unsigned)std::min<int64_t>(t->counters[kNStart], t->dev.maxTracklets);
    t->kernelUs[7] = (TPC_K5_FUSE_K6A && (float)nTotal / (32.0f * (float)t->k5Blocks) <= (float)(kK5PhasedThreads / 32)) ? 1.f : 0.f;
    return TPC_OK;
}

int tpc_get_tracks(tpc_tracker* t, const tpc_track** tracks, int32_t* n_tracks, const uint32_t** cluster_ids,
                   int64_t* n_cluster_ids) {
    if (!t || !tracks || !n_tracks || !cluster_ids || !n_cluster_ids) return TPC_E_ARG;
    int rc = tpc_sync(t);
    if (rc != TPC_OK) return rc;
    const int64_t nT = t->counters[kNTracks], nC = t->counters[kNTrackClusters];
    if (!t->fetched) {
        // "fetch the rest" only if the queued estimate was short
        const int64_t haveT = std::min(t->queuedTracks, nT), haveC = std::min(t->queuedIds, nC);
        if (haveT < nT || haveC < nC) {
            rc = ensure_out(t, nT, nC);
            if (rc != TPC_OK) return rc;
            if (haveT < nT) CUDA_TRY(t, cudaMemcpyAsync(t->outTracks + haveT, t->dev.tracks + haveT, sizeof(tpc_track) * (nT - haveT), cudaMemcpyDeviceToHost, t->stream));
            if (haveC < nC) CUDA_TRY(t, cudaMemcpyAsync(t->outIds + haveC, t->dev.clusterIds + haveC, sizeof(uint32_t) * (nC - haveC), cudaMemcpyDeviceToHost, t->stream));
            CUDA_TRY(t, cudaStreamSynchronize(t->stream));
            t->nRefetch++;
        }
        t->estTracks = nT + nT / 4 + 64; t->estIds = nC + nC / 4 + 1024;
    }
    *tracks = t->outTracks; *n_tracks = (int32_t)nT; *cluster_ids = t->outIds; *n_cluster_ids = nC;
    t->fetched = true;
    return t->counters[kNStart] > (uint32_t)t->dev.maxTracklets ? TPC_E_OVERFLOW : TPC_OK;
}

// PAPER.md:107 slicing: the event's sectors in groups, one group after the other through the same workspace.
int tpc_track_event_sliced(tpc_tracker* t, const int32_t* row_counts, const float* y, const float* z, int32_t sectors_per_slice,
                           const tpc_track** tracks, int32_t* n_tracks, const uint32_t** cluster_ids, int64_t* n_cluster_ids) {
    if (!t || !row_counts || !tracks || !n_tracks || !cluster_ids || !n_cluster_ids || sectors_per_slice < 1) return TPC_E_ARG;
    if (!t->ws) return TPC_E_STATE;
    std::vector<int64_t> secBase(t->nSec + 1, 0);     // clusters in front of each sector = its offset in y, z and in the ids
    for (int s = 0; s < t->nSec; s++) {
        int64_t n = 0;
        for (int r = 0; r < t->nRows; r++) {
            const int32_t c = row_counts[s * t->nRows + r];
            if (c < 0) return TPC_E_ARG;
            n += c;
        }
        secBase[s + 1] = secBase[s] + n;
    }
    if (secBase[t->nSec] > 0 && (!y || !z)) return TPC_E_ARG;
    if (secBase[t->nSec] > 0xFFFFFFFFll) return TPC_E_ARG;                       // ids are 32-bit
    for (int s0 = 0; s0 < t->nSec; s0 += sectors_per_slice)
        if (secBase[std::min(t->nSec, s0 + sectors_per_slice)] - secBase[s0] > t->maxClusters) return TPC_E_NOMEM;
    t->slTracks.clear(); t->slIds.clear();
    std::vector<int32_t> counts(t->nRowsTotal);
    for (int s0 = 0; s0 < t->nSec; s0 += sectors_per_slice) {
        const int s1 = std::min(t->nSec, s0 + sectors_per_slice);
        std::fill(counts.begin(), counts.end(), 0);
        std::copy(row_counts + (size_t)s0 * t->nRows, row_counts + (size_t)s1 * t->nRows, counts.begin() + (size_t)s0 * t->nRows);
        const int64_t base = secBase[s0];
        int rc = tpc_load_event(t, counts.data(), y ? y + base : nullptr, z ? z + base : nullptr);
        if (rc != TPC_OK) return rc;
        if ((rc = tpc_track_sectors(t)) != TPC_OK) return rc;
        const tpc_track* tr = nullptr; const uint32_t* ids = nullptr;
        int32_t nT = 0; int64_t nC = 0;
        if ((rc = tpc_get_tracks(t, &tr, &nT, &ids, &nC)) != TPC_OK) return rc;     // (waits for the slice: also for its input DMA)
        const int64_t idOff = (int64_t)t->slIds.size();
        if (idOff + nC > 0x7FFFFFFFll) return TPC_E_ARG;                         // cluster_offset is an int32
        const size_t tOff = t->slTracks.size();
        t->slTracks.resize(tOff + (size_t)nT);
        t->slIds.resize((size_t)(idOff + nC));
        if (nT) std::memcpy(t->slTracks.data() + tOff, tr, sizeof(tpc_track) * (size_t)nT);
        for (int32_t i = 0; i < nT; i++) t->slTracks[tOff + i].cluster_offset += (int32_t)idOff;
        uint32_t* dst = t->slIds.data() + idOff;
        for (int64_t i = 0; i < nC; i++) dst[i] = ids[i] + (uint32_t)base;
    }
    *tracks = t->slTracks.data(); *n_tracks = (int32_t)t->slTracks.size();
    *cluster_ids = t->slIds.data(); *n_cluster_ids = (int64_t)t->slIds.size();
    return TPC_OK;
}

int tpc_get_stats(tpc_tracker* t, tpc_stats* out) {
    if (!t || !out) return TPC_E_ARG;
    std::memset(out, 0, sizeof(*out));
    out->n_clusters = t->nClusters;
    out->max_clusters = t->maxClusters;
    out->max_tracklets = t->ws ? t->dev.maxTracklets : 0;
    out->workspace_bytes_used = (int64_t)t->L.total;
    out->n_output_refetches = t->nRefetch;
    if (t->refitFetched) out->refit_us = t->refitUs;
    if (t->mergeFetched) { out->merge_us = t->mergeUs; out->n_merged_tracks = t->nMerged; out->n_merge_links = t->nMergeLinks; }
    if (!t->tracked) return TPC_OK;
    out->n_links = t->counters[kNLinks];
    out->n_start_hits = t->counters[kNStart];
    out->n_tracklets = t->counters[kNKept];
    out->n_tracklet_hits = t->counters[kHitsTotal];
    out->n_tracks = t->counters[kNTracks];
    out->n_track_clusters = t->counters[kNTrackClusters];
    std::memcpy(out->kernel_us, t->kernelUs, sizeof(out->kernel_us));
    return TPC_OK;
}

size_t tpc_debug_dump_bytes(tpc_tracker* t, int stage) {
    if (!t || !t->tracked) return 0;
    if (tpc_sync(t) != TPC_OK) return 0;
    const size_t N = (size_t)t->nClusters;
    const size_t M = std::min<size_t>(t->counters[kNStart], (size_t)t->dev.maxTracklets);
    switch (stage) {
        case TPC_DUMP_LINKS: return 4 * N * sizeof(int32_t);
        case TPC_DUMP_START_HITS: return M * sizeof(uint32_t);
        case TPC_DUMP_TRACKLETS: return M * (sizeof(tpc_tracklet) + sizeof(int32_t) * t->nRows);
        case TPC_DUMP_OWNERS: return N * sizeof(uint32_t);
        default: return 0;
    }
}

int tpc_debug_dump(tpc_tracker* t, int stage, void* host_dst, size_t bytes) {
    if (!t || (!host_dst && bytes)) return TPC_E_ARG;
    if (!t->tracked) return TPC_E_STATE;
    const size_t need = tpc_debug_dump_bytes(t, stage);
    if (stage < TPC_DUMP_LINKS || stage > TPC_DUMP_OWNERS || bytes != need) return TPC_E_ARG;
    if (need == 0) return TPC_OK;
    const size_t N = (size_t)t->nClusters;
    const unsigned M = (unsigned)std::min<size_t>(t->counters[kNStart], (size_t)t->dev.maxTracklets);
    void* tmp = nullptr;
    cudaStream_t s = t->stream;
    int rc = TPC_OK;
    auto fail = [&](cudaError_t e) { t->lastCuda = (int)e; rc = TPC_E_CUDA; };
    cudaError_t e;
    if (stage == TPC_DUMP_TRACKLETS) {
        const size_t rhBytes = (size_t)M * t->nRows * sizeof(int32_t);
        if ((e = cudaMalloc(&tmp, rhBytes)) != cudaSuccess) { fail(e); return rc; }
        dump_rowhit_kernel<<<M, 64, 0, s>>>(t->dev, t->nRows, M, (int32_t*)tmp);
        std::vector<TrackletRec> recs(M);
        if ((e = cudaMemcpyAsync(recs.data(), t->dev.recs, sizeof(TrackletRec) * M, cudaMemcpyDeviceToHost, s)) != cudaSuccess) fail(e);
        char* dst = (char*)host_dst;
        if (rc == TPC_OK && (e = cudaMemcpyAsync(dst + sizeof(tpc_tracklet) * M, tmp, rhBytes, cudaMemcpyDeviceToHost, s)) != cudaSuccess) fail(e);
        if ((e = cudaStreamSynchronize(s)) != cudaSuccess) fail(e);
        if (rc == TPC_OK) {
            tpc_tracklet* o = (tpc_tracklet*)dst;
            for (unsigned i = 0; i < M; i++) {
                const TrackletRec& r = recs[i];
                o[i].start_gid = r.startGid; o[i].sector = r.sector; o[i].start_row = r.startRow; o[i].n_hits = r.nHits;
                o[i].first_row = r.firstRow; o[i].last_row = r.lastRow; o[i].n_fit = r.nFit;
                o[i].x = (r.xRow >= 0 && r.xRow < t->nRows) ? t->rowX[r.xRow] : 0.f;
                std::memcpy(o[i].p, r.p, sizeof(r.p)); std::memcpy(o[i].c, r.c, sizeof(r.c)); o[i].chi2 = r.chi2;
            }
        }
    } else {
        if ((e = cudaMalloc(&tmp, need)) != cudaSuccess) { fail(e); return rc; }
        if (stage == TPC_DUMP_LINKS) dump_links_kernel<<<t->nRowsTotal, 128, 0, s>>>(t->dev, t->nRows, (int64_t)N, (int32_t*)tmp);
        else if (stage == TPC_DUMP_START_HITS) dump_starts_kernel<<<(M + 127) / 128, 128, 0, s>>>(t->dev, M, (uint32_t*)tmp);
        else dump_owner_kernel<<<t->nRowsTotal, 128, 0, s>>>(t->dev, t->nRows, (uint32_t*)tmp);
        if ((e = cudaMemcpyAsync(host_dst, tmp, need, cudaMemcpyDeviceToHost, s)) != cudaSuccess) fail(e);
        if ((e = cudaStreamSynchronize(s)) != cudaSuccess) fail(e);
    }
    if ((e = cudaGetLastError()) != cudaSuccess) fail(e);
    cudaFree(tmp);
    return rc;
}

int tpc_debug_check_guards(tpc_tracker* t) {
    if (!t) return TPC_E_ARG;
    if (!t->ws) return TPC_E_STATE;
    CUDA_TRY(t, cudaStreamSynchronize(t->stream));
    std::vector<unsigned char> h(kAlign);
    int bad = 0;
    for (int g = 0; g < t->L.nGuards; g++) {
        CUDA_TRY(t, cudaMemcpy(h.data(), t->ws + t->L.guard[g], kAlign, cudaMemcpyDeviceToHost));
        for (unsigned char c : h) if (c != 0xA5) { bad++; break; }
    }
    return bad;      // number of guard zones that were written to
}

const char* tpc_strerror(int code) {
    switch (code) {
        case TPC_OK: return "ok";
        case TPC_E_ARG: return "invalid argument";
        case TPC_E_STATE: return "call out of order";
        case TPC_E_NOMEM: return "workspace too small";
        case TPC_E_OVERFLOW: return "tracklet capacity exceeded";
        case TPC_E_CUDA: return "CUDA error or no device";
        case TPC_E_LIMIT: return "more tracks or (sector,row) bins than the fixed scratch of tpc_merge_links_no_alloc holds";
        default: return "unknown error";
    }
}

int tpc_last_cuda_error(const tpc_tracker* t) { return t ? t->lastCuda : 0; }

}  // extern "C"

// ------------------------------------------------------------------------------------------ K7 without allocation
// tpc_merge_links_no_alloc (tpctrk.h): the K7 kernels of tpc_merge_tracks on caller-owned tracks and outputs, their
// scratch in the file-scope array below instead of a tracker workspace.  Nothing here allocates.
namespace {

constexpr size_t kNaMaxT = TPC_NO_ALLOC_MAX_TRACKS, kNaMaxB = TPC_NO_ALLOC_MAX_BINS;
constexpr size_t na_up(size_t v) { return (v + kAlign - 1) / kAlign * kAlign; }
// sections of the scratch array [bytes from its start], each a multiple of 256
constexpr size_t kNaCounters = 0;                                              // uint32[kNCounters]: [kNTracks] = n_tracks
constexpr size_t kNaMCount = kNaCounters + na_up(sizeof(uint32_t) * kNCounters);   // uint32[2] (k7_init clears it)
constexpr size_t kNaKey = kNaMCount + kAlign;                                  // uint32[maxT]
constexpr size_t kNaOrder = kNaKey + na_up(sizeof(uint32_t) * kNaMaxT);     // uint32[maxT]
constexpr size_t kNaBestIn = kNaOrder + na_up(sizeof(uint32_t) * kNaMaxT);  // uint64[maxT]
constexpr size_t kNaOut = kNaBestIn + na_up(sizeof(unsigned long long) * kNaMaxT);   // int32[maxT]
constexpr size_t kNaOutChi2 = kNaOut + na_up(sizeof(int32_t) * kNaMaxT);    // float[maxT]
constexpr size_t kNaBinStart = kNaOutChi2 + na_up(sizeof(float) * kNaMaxT); // uint32[maxB + 2]
constexpr size_t kNaBinCursor = kNaBinStart + na_up(sizeof(uint32_t) * (kNaMaxB + 2));   // uint32[maxB + 1]
constexpr size_t kNaBytes = kNaBinCursor + na_up(sizeof(uint32_t) * (kNaMaxB + 1));
static_assert(kNaBytes < (2u << 20), "the no-allocation scratch is meant to stay modest (tpctrk.h says about 1.7 MB)");

}  // namespace

// In host code this name is a stand-in for the symbol, not a device address: kernels get the pointer that
// cudaGetSymbolAddress returns for the current device (na_device below); device code may name the array directly.
static __device__ __align__(256) unsigned char g_k7NaScratch[kNaBytes];

namespace {

// the track count where the K7 kernels look for it, the other counters zero (device code: names the array itself)
__global__ void k7na_begin(int nTracks) {
    uint32_t* c = reinterpret_cast<uint32_t*>(g_k7NaScratch + kNaCounters);
    if (threadIdx.x < kNCounters) c[threadIdx.x] = threadIdx.x == kNTracks ? (uint32_t)nTracks : 0u;
}

struct NaDevice { unsigned char* scratch = nullptr; int blocks = 0; };
constexpr int kNaMaxDevices = 64;
NaDevice g_naDev[kNaMaxDevices];
std::mutex g_naLock;

// Once per device, with that device current: the device address of the scratch array and the grid of the K7 kernels.
cudaError_t na_device(int dev, NaDevice& out) {
    std::lock_guard<std::mutex> lk(g_naLock);
    NaDevice& d = g_naDev[dev];
    if (!d.scratch) {
        void* p = nullptr;
        cudaError_t e = cudaGetSymbolAddress(&p, g_k7NaScratch);
        if (e != cudaSuccess) return e;
        int sms = 0, occ = 0;
        if ((e = cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev)) != cudaSuccess) return e;
        if ((e = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, k7_match, kK7Threads, 0)) != cudaSuccess) return e;
        d.blocks = std::max(1, sms) * std::max(1, occ);
        d.scratch = static_cast<unsigned char*>(p);
    }
    out = d;
    return cudaSuccess;
}

}  // namespace

extern "C" int tpc_merge_links_no_alloc(int32_t n_sectors, int32_t n_rows, float sector_dphi, float bz_tesla, const tpc_params* params,
                                        const tpc_track* dev_tracks, int32_t n_tracks, const uint32_t* dev_cluster_ids,
                                        int32_t* dev_next, int32_t* dev_prev, float* dev_chi2, void* cuda_stream, int* cuda_error) {
    if (cuda_error) *cuda_error = 0;
    auto cuda_fail = [&](cudaError_t e) { if (cuda_error) *cuda_error = (int)e; return (int)TPC_E_CUDA; };
    if (n_sectors < 1 || n_rows < 3 || n_rows > kMaxRows || n_tracks < 0) return TPC_E_ARG;
    if ((int64_t)n_sectors * n_rows > (int64_t)kNaMaxB || (int64_t)n_tracks > (int64_t)kNaMaxT) return TPC_E_LIMIT;
    if (n_tracks > 0 && (!dev_tracks || !dev_cluster_ids || !dev_next || !dev_prev || !dev_chi2)) return TPC_E_ARG;
    tpc_params P;
    if (params) P = *params; else tpc_default_params(&P);
    if (!(P.kf_smax > 0.f && P.kf_smax < 1.f) || !(P.merge_chi2 >= 0.f && P.merge_chi2 < 1e30f) || P.merge_max_row_gap < 0 ||
        !(std::abs(bz_tesla) < 1e3f) || !(std::abs(sector_dphi) < 1e3f)) return TPC_E_ARG;
    int dev = -1;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) return cuda_fail(e);
    if (dev < 0 || dev >= kNaMaxDevices) return TPC_E_ARG;
    NaDevice nd;
    if ((e = na_device(dev, nd)) != cudaSuccess) return cuda_fail(e);
    if (n_tracks == 0) return TPC_OK;

    MergePtrs m{};
    m.tracks = dev_tracks; m.clusterIds = dev_cluster_ids;
    m.counters = reinterpret_cast<const uint32_t*>(nd.scratch + kNaCounters);
    m.mcount = reinterpret_cast<uint32_t*>(nd.scratch + kNaMCount);
    m.key = reinterpret_cast<uint32_t*>(nd.scratch + kNaKey);
    m.order = reinterpret_cast<uint32_t*>(nd.scratch + kNaOrder);
    m.bestIn = reinterpret_cast<unsigned long long*>(nd.scratch + kNaBestIn);
    m.out = reinterpret_cast<int32_t*>(nd.scratch + kNaOut);
    m.outChi2 = reinterpret_cast<float*>(nd.scratch + kNaOutChi2);
    m.binStart = reinterpret_cast<uint32_t*>(nd.scratch + kNaBinStart);
    m.binCursor = reinterpret_cast<uint32_t*>(nd.scratch + kNaBinCursor);
    m.next = dev_next; m.prev = dev_prev; m.chi2 = dev_chi2;
    m.merged = nullptr; m.segments = nullptr;        // k7_chains is not part of this entry point: the links are the result
    m.nBins = n_sectors * n_rows;
    DevParams dp; dp.P = P; dp.CB = (float)(-0.299792458e-2 * (double)bz_tesla); dp.nSec = n_sectors; dp.nRows = n_rows;
    const int perSide = n_sectors >= 36 ? 18 : n_sectors;
    const float cosB = (float)std::cos((double)sector_dphi), sinB = (float)std::sin((double)sector_dphi);
    cudaStream_t s = static_cast<cudaStream_t>(cuda_stream);
    const int grid = nd.blocks;
    k7na_begin<<<1, 32, 0, s>>>(n_tracks);
    k7_init<<<grid, kK7Threads, 0, s>>>(m, n_rows);        // clears the bins, the cursors, the best-partner words, the outputs
    k7_hist<<<grid, kK7Threads, 0, s>>>(m, n_rows);
    k7_scan<<<1, 1024, 0, s>>>(m);
    k7_scatter<<<grid, kK7Threads, 0, s>>>(m, n_rows);
    k7_match<<<grid, kK7Threads, 0, s>>>(m, dp, perSide, cosB, sinB);
    k7_link<<<grid, kK7Threads, 0, s>>>(m);
    if ((e = cudaGetLastError()) != cudaSuccess) return cuda_fail(e);
    return TPC_OK;
}
