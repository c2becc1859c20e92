// Device-side data layout of the tracker.
#pragma once
#include <cstdint>
#include <cuda_runtime.h>

#include "tpctrk.h"

namespace tpc {

constexpr int kMaxRows = 255;          // n_rows limit: nHits must fit the 8-bit field of the ownership key
constexpr int kRowPad = 4;             // a row's sorted hits start at a multiple of 4 hits (32 B sector, 16 B TMA)
constexpr int kMaxBinsPerRow = 8192;   // K1 histogram lives in shared memory (32 KB)
constexpr float kGridMargin = 1e-3f;   // [cm] slack of every bin-range query; the exact window test follows

// One (sector,row), hot part: exactly the eight words a grid query needs (two 16-byte loads, no dead lanes:
// a partly-used vector load makes the unused destination registers a write-after-write hazard for whatever the
// compiler puts there next, which serialises the "prefetched" load).  Host fills hitOff/binOff; K1 fills the grid.
struct __align__(32) RowGrid {
    int32_t hitOff;    // offset of the row's sorted hits in hits[]/orig[]/links/weight (multiple of kRowPad)
    int32_t binOff;    // offset of the row's binStart[nBins+1] / buckets[nBins]
    int32_t nY, nZ;    // grid dimensions (K1; 1x1 with an empty bucket for an empty row)
    float y0, z0;      // grid origin (K1)
    float invY, invZ;  // 1 / bin size (K1)
};
static_assert(sizeof(RowGrid) == 32, "RowGrid layout");

// One (sector,row), cold part (host-filled).
struct __align__(16) RowMeta {
    int32_t n;         // clusters in the row
    int32_t inOff;     // offset of the row's clusters in the staging arrays, as loaded
    uint32_t gidBase;  // event-global id of load index 0 (canonical ids)
    int32_t maxBins;   // capacity reserved for this row's bins
};
static_assert(sizeof(RowMeta) == 16, "RowMeta layout");

// One grid bin, one 32-byte sector: where the bin's hits start in the sorted arrays, how many there are, and the
// first three of them inline, so that a road search costs ONE dependent memory level instead of two
// (binStart -> hits).  Bins with more than three hits continue in hits[start+3 ...].
struct __align__(32) Bucket {
    uint32_t start, count;
    float2 h[3];
};
static_assert(sizeof(Bucket) == 32, "Bucket layout");

// Per-tracklet record written by K5 (128 B, float4-aligned).
struct __align__(16) TrackletRec {
    uint32_t startGid;
    int32_t sector, startRow, nHits, firstRow, lastRow, nFit, xRow;
    float p[5];
    float c[15];
    float chi2;
    uint32_t ownerKey;     // K6's ownership key (S6), written by K5 with the record
    float pad[2];
};
static_assert(sizeof(TrackletRec) == 128, "TrackletRec layout");

// Programmatic dependent launch (tpctrk.cu launches K2..K6 as dependents of the kernel before them when no CUDA events
// sit between the kernels): grid_dep_wait() returns when the preceding kernel has completed and its writes are
// visible; every thread of every dependent kernel calls it on every path before it reads anything an earlier kernel
// of the call wrote and before it exits, so that "this kernel has completed" keeps implying "all earlier ones have".
// A no-op for a kernel launched the ordinary way.  grid_dep_trigger(): the dependent kernel may start its prologue.
#ifndef TPC_PDL_TRIGGER
#define TPC_PDL_TRIGGER 1
#endif
__device__ __forceinline__ void grid_dep_wait() { asm volatile("griddepcontrol.wait;" ::: "memory"); }
__device__ __forceinline__ void grid_dep_trigger() { asm volatile("griddepcontrol.launch_dependents;" ::: "memory"); }

struct DevParams {
    tpc_params P;
    float CB;          // curvature per unit q/pT: kappa = p[4]*CB  [1/cm per c/GeV]
    int32_t nSec, nRows;
};

enum Counter { kNStart = 0, kQueue = 1, kNTracks = 2, kNTrackClusters = 3 /* = kNTracks + 1, 8-byte aligned pair (K6b) */, kNKept = 4, kHitsTotal = 5, kNLinks = 6, kWarpsDone = 7 /* phased K5: warps that have finished their tracklets */,
               kNPending = 8 /* ... and how many of them left their K6a weights pass to the k6_weights launch */, kNCounters = 16 };
// counters[kNCounters + i], i < kMaxPending: the groups of 32 tracklet slots whose weights pass is still to do
enum : int { kMaxPending = 4096 };

// All device pointers of one tracker; passed by value to the kernels.
struct DevPtrs {
    const float* inY;
    const float* inZ;
    RowGrid* grid;         // [nRowsTotal]
    const RowMeta* meta;   // [nRowsTotal]
    const float* rowX;
    float2* hits;          // sorted (y,z) pairs
    uint32_t* orig;        // sorted position -> event-global cluster id (gidBase of the row + load index)
    uint32_t* binStart;
    Bucket* buckets;       // [binCap], same indexing as binStart (row.binOff + bin)
    int32_t* linkUp;       // raw links, index = sorted position in the adjacent row
    int32_t* linkDn;
    int32_t* linkUpC;      // cleaned links
    int32_t* linkDnC;
    uint32_t* weight;      // ownership key per hit
    int4* startsRaw;       // K3/K4 output in append order: (rowId, sorted position, sorted position of the linked hit in the
                           // row above, global id); read by the free-running K5 kernel
    int4* starts;          // the same records filed by pad row: row r's start hits at starts[rowStartBase[r] + 0..rowHist[r]);
                           // read by the phased K5 kernel, which wants a warp's tracklets to start in the same row
    uint32_t* rowHist;     // [kMaxRows + 1] start hits per pad row (K3/K4 atomics)
    const uint32_t* rowStartBase;   // [kMaxRows + 2] host: exclusive prefix over rows of the clusters per row (all sectors) =
                                    // where row r's segment of starts[] begins (a row has at most as many start hits as hits)
    TrackletRec* recs;
    int32_t* rowHit;       // [maxTracklets][rhStride], GLOBAL sorted position (row hitOff + position) of the tracklet's hit
                           // in each row, -1 none: indexes weight[] / orig[] directly
    tpc_track* tracks;
    uint32_t* clusterIds;
    uint32_t* clusterPos;  // same order as clusterIds: global sorted position of the cluster (hits[] holds its y, z) ...
    uint8_t* clusterRow;   // ... and its pad row: what the final fit (K8) reads
    uint32_t* counters;
    uint32_t* sectorGidBase;
    int32_t nRowsTotal;
    int32_t maxTracklets;
    int32_t rhStride;      // n_rows rounded up to a multiple of 32
};

}  // namespace tpc
