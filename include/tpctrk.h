/*
 * tpctrk.h — C ABI of the B200-native Phase-I TPC sector tracker (libtpctrk.so).
 *
 * The calls follow the paper's statement of the problem (arxiv 1712.09430; PAPER.md = /root/reference/PAPER.md):
 *   clusters (x,y,z) per TPC sector and pad row
 *     -> Phase I, step 1: cellular-automaton seeding, one GPU thread per hit
 *     -> Phase I, step 2: track following with a simplified Kalman filter, one thread per track
 *        candidate, and selection of the best instance per track segment
 *     -> tracklets with cluster lists and 5-parameter states plus covariances.
 * The numerical readings (S0..S6, R-1..R-15) are listed in DESIGN.md.
 *
 * Conventions
 *  - Plain C, no exceptions or aborts cross the ABI.  Every int-returning call returns TPC_OK (0) or a
 *    negative tpc_error; tpc_strerror() names it.
 *  - "device pointer" = CUDA device memory of the current device; "host pointer" = ordinary or pinned host
 *    memory.  Where a call accepts either, the kind is detected with cudaPointerGetAttributes.
 *  - All work is enqueued on the stream given to tpc_set_stream (default: the legacy default stream).
 *    Calls are asynchronous unless stated otherwise.
 *  - The library never allocates device memory for the hot path: the caller hands it one workspace
 *    (tpc_set_workspace), e.g. a torch tensor, and keeps ownership.  Pinned host memory for result
 *    download is library-owned.
 *  - There is no CPU fallback: without a CUDA device every compute call returns TPC_E_CUDA.
 */
#ifndef TPCTRK_H
#define TPCTRK_H

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct tpc_tracker tpc_tracker; /* opaque, library-owned */

typedef enum tpc_error {
    TPC_OK = 0,
    TPC_E_ARG = -1,      /* null pointer, sector/row/count out of range, unsupported geometry */
    TPC_E_STATE = -2,    /* call out of order (no workspace, nothing loaded, nothing tracked yet) */
    TPC_E_NOMEM = -3,    /* workspace too small for the loaded clusters; see tpc_workspace_bytes */
    TPC_E_OVERFLOW = -4, /* tracklet-capacity estimate exceeded ("estimation was too small");
                            tpc_stats.n_start_hits holds the required capacity; enlarge and re-run */
    TPC_E_CUDA = -5,     /* CUDA runtime error or no device; tpc_last_cuda_error() has the code */
    TPC_E_LIMIT = -6     /* tpc_merge_links_no_alloc: more tracks or (sector,row) bins than its fixed scratch holds */
} tpc_error;

/* Constants of the method (the paper gives none). */
typedef struct tpc_params {
    float err2_y, err2_z;           /* measurement variances [cm^2], uncorrelated          0.01 */
    float nf_ty, nf_tz;             /* neighbour window slope limits |dy/dx|, |dz/dx|  1.0, 1.5 */
    float nf_c;                     /* neighbour window padding [cm]                                      0.5 */
    float nf_d2max;                 /* max squared 3-point collinearity residual [cm^2]                  0.25 */
    float kf_css0, kf_ctt0, kf_ckk0;/* initial variances of sin(phi), dz/ds, q/pT                  1, 10, 100 */
    float kf_smax;                  /* propagation fails for |sin(phi)| >= this            0.95 */
    float road_nsig, road_max;      /* search road = min(road_max, nsig*sqrt(C+err2)) per coordinate   4, 2.0 */
    int32_t max_gap;                /* a leg stops at the (max_gap+1)-th consecutive empty row              4 */
    int32_t min_hits;               /* min hits of a kept tracklet and min owned hits of a track           10 */
    int32_t seed_min_chain;         /* min link-chain length of a seed ("3 to about 10")        3 */
    float max_tracklets_per_cluster;/* capacity estimate for tracklets                      0.1 */
    float grid_bins_per_hit;        /* resolution of the per-row y/z grid (accelerator only: no result
                                       depends on it), bins per cluster of the row, 0.25..64                2 */
    float merge_chi2;               /* Phase II merging: max chi2 (5 parameters) of two matching segments  50 */
    int32_t merge_max_row_gap;      /* ... max pad rows between the end of the inner segment and the
                                       start of the outer one                                              40 */
    float field_ar, field_az;       /* final fit: Bz(r, z) = Bz (1 + field_ar r^2 + field_az z^2), the polynomial
                                       field approximation of PAPER.md:46  [1/cm^2]                       0, 0 */
    float ms_x0_inv;                /* final fit: 1 / radiation length of the gas [1/cm]; 0 = no multiple
                                       scattering noise                                                     0 */
} tpc_params;

typedef struct tpc_geometry {
    int32_t n_sectors;        /* 36: s<18 side A (z>0), s>=18 side C (z<0); any value >= 1 works */
    int32_t n_rows;           /* 159 pad rows; 3 <= n_rows <= 255 */
    const float* row_x;       /* host pointer, n_rows ascending pad-row x [cm]; copied at create */
    float sector_dphi;        /* angle between the frames of neighbouring sectors [rad] (20 deg); Phase I is sector-local
                                 and does not use it, tpc_merge_tracks rotates states by it */
    float z_max;              /* informational: drift length [cm] */
    const tpc_params* params; /* host pointer or NULL = defaults */
} tpc_geometry;

/* One output track = one selected tracklet.  State is given at x (sector-local frame):
 * p = (y, z, sin(phi), dz/ds, q/pT); c = lower triangle yy, zy,zz, sy,sz,ss, ty,tz,ts,tt, ky,kz,ks,kt,kk. */
typedef struct tpc_track {
    int32_t sector, n_clusters, first_row, last_row;
    int32_t cluster_offset;   /* into cluster_ids; ids ascending in row, one per row */
    float x;
    float p[5];
    float c[15];
    float chi2;
    int32_t n_fit;            /* number of hit updates in the final (inward) filter pass */
} tpc_track;

/* Counters and device times of the last tpc_track_sectors (valid after tpc_get_tracks / tpc_sync). */
typedef struct tpc_stats {
    int64_t n_clusters, n_links, n_start_hits, n_tracklets, n_tracklet_hits, n_tracks, n_track_clusters;
    int64_t workspace_bytes_used, max_clusters, max_tracklets;
    int64_t n_output_refetches; /* calls of tpc_get_tracks (since create) that had to fetch a remainder because the
                                 download queued by tpc_track_sectors was estimated too small */
    float merge_us;           /* device time of the last tpc_merge_tracks (K7), valid after tpc_get_merged */
    int32_t n_merged_tracks, n_merge_links;   /* after tpc_get_merged */
    float refit_us;           /* device time of the last tpc_refit_tracks (K8), valid after tpc_get_refit */
    float kernel_us[8];       /* K1 sort+grid, K2 neighbours, K3/K4 clean+start, K5 construct, K6a weights,
                                 K6b select+compact, [6] = K1..K6 total, [7] = 1.0 if the K6a weights pass of this
                                 event ran inside the K5 launch (about one tracklet per GPU thread or fewer: [3]
                                 then includes it and [4] only covers the few tracklets the last K5 warps left over), else 0.0 */
} tpc_stats;

/* Record of tpc_debug_dump(TPC_DUMP_TRACKLETS). */
typedef struct tpc_tracklet {
    uint32_t start_gid;       /* event-global id of the start hit = canonical tracklet id */
    int32_t sector, start_row, n_hits, first_row, last_row, n_fit;
    float x, p[5], c[15], chi2;
} tpc_tracklet;

enum {
    TPC_DUMP_LINKS = 1,       /* int32[4][N]: linkUp, linkDn after K2; linkUp, linkDn after K3.  Indexed by global id;
                                 value = LOAD index of the linked hit inside row r+1 / r-1, -1 none */
    TPC_DUMP_START_HITS = 2,  /* uint32[n_start_hits]: global ids, unordered */
    TPC_DUMP_TRACKLETS = 3,   /* tpc_tracklet[n_start_hits] then int32[n_start_hits][n_rows] row->load index, -1 none */
    TPC_DUMP_OWNERS = 4       /* uint32[N]: start_gid of the owning tracklet, 0xFFFFFFFF none */
};

/* Defaults of DESIGN.md "Constants". */
void tpc_default_params(tpc_params* p);

/* Create a tracker for a geometry and a constant field Bz [T].  g and its pointers are host
 * memory, copied.  *out is owned by the library until tpc_tracker_destroy.  Does not touch the GPU.
 * TPC_E_ARG for an unsupported geometry and for parameters outside their domain: variances (err2_*, kf_c**0),
 * road_nsig, road_max and max_tracklets_per_cluster must be positive and finite, kf_smax inside (0,1), the nf_* window
 * constants non-negative, min_hits >= 1, max_gap >= 0, seed_min_chain >= 2, grid_bins_per_hit in [0.25, 64]. */
int tpc_tracker_create(const tpc_geometry* g, float bz_tesla, tpc_tracker** out);
void tpc_tracker_destroy(tpc_tracker* t);

/* cuda_stream: a cudaStream_t (e.g. torch.cuda.current_stream().cuda_stream); NULL = default stream. */
int tpc_set_stream(tpc_tracker* t, void* cuda_stream);

/* Per-kernel times in tpc_stats.kernel_us[0..5]: on != 0 records a CUDA event between the kernels of every
 * tpc_track_sectors.  Off by default: without the events K2..K6 are launched as programmatic dependents of the
 * kernel before them (a kernel's launch, and K5's shared-memory prologue, overlap the end of the previous kernel),
 * which the event records prevent: ~30 us per call (5 % of a central event).  kernel_us[6] (K1..K6 total) is always
 * measured; with the timing off kernel_us[0..5] are 0.  Results are identical either way. */
int tpc_set_kernel_timing(tpc_tracker* t, int on);

/* on != 0 (default): K2..K6 are launched as programmatic dependents of the kernel before them (only possible while
 * the kernel timing is off): -15 us per central event for a tracker that has the GPU to itself.  With several
 * trackers on concurrent streams it makes little difference either way (end to end, one host thread: 0.51 vs 0.51 ms
 * per event with six trackers in flight, 0.51 vs 0.55 with four). */
int tpc_set_dependent_launch(tpc_tracker* t, int on);

/* on != 0: the neighbours finder (K2) stages the pieces of the two adjacent pad rows that a block's hits can reach
 * in shared memory (bulk copies by the TMA engine) before it scans them; off (default): it reads them through L1.
 * A launch option like the two above: results are identical.  Off is faster on B200 for every workload measured
 * (central event 90 vs 120 us, time frame 10.0 vs 11.4 ms; profiles/r02_k2_staging.md). */
int tpc_set_neighbour_staging(tpc_tracker* t, int on);

/* Device bytes needed for events of up to max_clusters clusters (internal buffers). */
size_t tpc_workspace_bytes(const tpc_tracker* t, int64_t max_clusters);
/* dev_ptr: device pointer, 256-byte aligned, caller-owned, must outlive its use.  Capacity is derived from bytes. */
int tpc_set_workspace(tpc_tracker* t, void* dev_ptr, size_t bytes);

/* Forget all loaded clusters. */
int tpc_reset_event(tpc_tracker* t);

/* Load the n clusters of one (sector,row).  x, y, z: n floats each, all host or all device pointers; copied
 * (device: enqueued on the stream; host: staged in pinned memory, uploaded by tpc_track_sectors).  x may be NULL and
 * is not used: the tracker takes the pad-row x (R-13).  Index i in this call is the cluster's load index;
 * its event-global id is rowBase(sector,row)+i with rowBase the exclusive prefix sum of the loaded counts in
 * ascending (sector,row) order.  Loading a (sector,row) again replaces it: in place if the new load is not larger than
 * the largest earlier load of that (sector,row) since the last reset, otherwise appended - the old staging slots then
 * count against max_clusters until tpc_reset_event.
 * Returns TPC_E_NOMEM when the staging area is full.  Non-finite coordinates give undefined tracks but never a crash
 * or hang. */
int tpc_load_clusters(tpc_tracker* t, int sector, int row, int n, const float* x, const float* y, const float* z);

/* Load a whole event at once: row_counts[n_sectors*n_rows] on the host; y, z concatenated in ascending (sector,row)
 * order, both host or both device pointers.  Replaces everything loaded before.
 * Ownership of y, z: ordinary host memory and device memory are copied (or the copy is ordered on the stream) before
 * the call returns.  PAGE-LOCKED host memory of 64 Ki clusters or more is read by DMA directly and the call returns
 * as soon as that copy is QUEUED (DMA runs beside the kernels): the buffers must stay untouched until
 * tpc_wait_input, tpc_sync or tpc_get_tracks has returned.  The same holds for tpc_load_clusters. */
int tpc_load_event(tpc_tracker* t, const int32_t* row_counts, const float* y, const float* z);

/* Block until every input buffer handed to tpc_load_clusters / tpc_load_event so far has been read. */
int tpc_wait_input(tpc_tracker* t);

/* Run K1..K6 (sort+grid, neighbours finder, cleaner+start hits, tracklet constructor, selector+compaction) on the
 * stream.  Asynchronous.  May be called repeatedly on the same loaded event.
 * Output of unknown size ("the tracker can estimate a buffer that is large enough to store all tracks
 * and queue the transfer of this buffer immediately ... if the estimation was too small, the tracker can still
 * fetch the rest"): behind K6 the call queues the download of the counters and of an estimated prefix of the tracks
 * and cluster ids (first event: one track per 64 clusters and one id per cluster; afterwards the last fetched
 * event's counts + 25 %) into library-owned pinned memory.  tpc_set_output_prefetch(t, 0) queues the counters only. */
int tpc_track_sectors(tpc_tracker* t);
int tpc_set_output_prefetch(tpc_tracker* t, int on);

/* Wait (once, on an event behind the queued download; the stream may hold later work) and hand out the result in
 * library-owned pinned memory (valid until the next track/reset/destroy).  Copies only the remainder, if the queued
 * estimate was short (tpc_stats.n_output_refetches counts those calls).
 * tracks[i].cluster_offset indexes cluster_ids (event-global ids).  Track order is unspecified.
 * Returns TPC_E_OVERFLOW if the tracklet capacity was exceeded (results then cover the first max_tracklets seeds). */
int tpc_get_tracks(tpc_tracker* t, const tpc_track** tracks, int32_t* n_tracks,
                   const uint32_t** cluster_ids, int64_t* n_cluster_ids);

/* Wait for the last tpc_track_sectors and its queued download; counters + per-kernel device times only. */
int tpc_sync(tpc_tracker* t);
int tpc_get_stats(tpc_tracker* t, tpc_stats* out);

/* ---- Phase II, first step: track merging (Table 1 "Matching Covariance"; reading S7 of DESIGN.md) ----
 * A merged track = a chain of Phase-I tracks ("segments") of one TPC side, each continued outward by the segment in
 * the same or a neighbouring sector that starts within merge_max_row_gap pad rows above its end and whose state is
 * nearest in chi2 (<= merge_chi2) after the inner state has been rotated into the outer segment's sector frame and
 * propagated to its x; a link is kept only if it is the best one from both ends.  Sectors s and s+1 (mod 18 within
 * a side; n_sectors < 36: one ring of all sectors) are neighbours, sector s+1's frame is sector s's turned by
 * +sector_dphi.  Parameters are those of the segments (no refit: PAPER.md:46 is a later step). */
typedef struct tpc_merged_track {
    int32_t n_segments;       /* 1 = a Phase-I track nothing was merged with */
    int32_t n_clusters;       /* sum over the segments */
    int32_t segment_offset;   /* into segments[]: track indices (as in tpc_get_tracks), innermost segment first */
    int32_t first_track;      /* = segments[segment_offset] */
} tpc_merged_track;

/* Run the merging kernels (K7) on the tracks of the last tpc_track_sectors, on the stream.  Asynchronous.
 * TPC_E_STATE before tpc_track_sectors. */
int tpc_merge_tracks(tpc_tracker* t);

/* Synchronise and download.  next[i] / prev[i]: index of the segment that continues track i outward / inward, -1
 * none; chi2[i]: chi2 of the link i -> next[i] (0 without link); n_tracks entries each, indexed like the arrays of
 * tpc_get_tracks of the same event.  merged[n_merged] in unspecified order, segments[n_tracks].  Library-owned
 * pinned memory, valid until the next merge/track/reset/destroy.  Any output pointer may be NULL. */
int tpc_get_merged(tpc_tracker* t, const int32_t** next, const int32_t** prev, const float** chi2, int32_t* n_tracks,
                   const tpc_merged_track** merged, int32_t* n_merged, const int32_t** segments);

/* ---- Phase II, second step: final fit of the merged tracks (reading S8 of DESIGN.md) ----
 * "the full track is refit using the full Kalman filter.  A polynomial approximation of the magnetic field avoids the
 * slow memory access to a field map."  One inward filter pass over ALL clusters of a merged track, from its outermost
 * cluster (the starting point) to its innermost one, across the sector frames of its segments; per step the field is
 * the polynomial of tpc_params at the state's point, and multiple scattering over the step's path is added to the
 * covariance (ms_x0_inv).  ok = 0: the pass could not be completed (|sin phi| limit); the record then repeats the
 * innermost segment's Phase-I state with n_fit = 0. */
typedef struct tpc_refit_track {
    int32_t first_track;      /* innermost segment (track index as in tpc_get_tracks) = tpc_merged_track.first_track */
    int32_t sector;           /* frame of the state */
    int32_t n_fit;            /* clusters used as measurements (all but the outermost one) */
    int32_t ok;
    float x, p[5], c[15], chi2;
} tpc_refit_track;

/* Run the final fit (K8) on the merged tracks of the last tpc_merge_tracks, on the stream.  Asynchronous.
 * TPC_E_STATE before tpc_merge_tracks. */
int tpc_refit_tracks(tpc_tracker* t);
/* Synchronise and download: refit[i] belongs to merged[i] of tpc_get_merged (same event).  Library-owned pinned memory. */
int tpc_get_refit(tpc_tracker* t, const tpc_refit_track** refit, int32_t* n_merged);

/* ---- Slicing ("If GPU memory would become insufficient, we can easily employ a slicing approach,
 * processing parts of the time-frame one after another in a similar fashion as we currently process the TPC sectors") ----
 * Phase I of a whole event (arguments as tpc_load_event: host or device pointers) in slices of sectors_per_slice
 * consecutive sectors, one slice after the other through the SAME workspace, which therefore only has to hold the
 * fullest slice: tpc_workspace_bytes(t, max over slices of the slice's clusters).  Sectors are independent in Phase I,
 * so the result is the unsliced one: the same tracks (sector numbers of the whole event, event-global cluster ids),
 * slice after slice.  Synchronous; the outputs are library-owned host memory, valid until the next sliced call or
 * destroy.  Afterwards the tracker holds the LAST slice (tpc_get_stats, tpc_debug_dump, tpc_merge_tracks see that
 * slice only; merging over all slices: upload the tracks and use tpc_merge_links_no_alloc, or run unsliced).
 * Errors: TPC_E_ARG (null pointer, negative count, sectors_per_slice < 1), TPC_E_STATE (no workspace), TPC_E_NOMEM (a
 * slice has more clusters than the workspace holds: checked before anything runs), TPC_E_OVERFLOW (a slice exceeded
 * the tracklet capacity: enlarge the workspace or take fewer sectors per slice). */
int tpc_track_event_sliced(tpc_tracker* t, const int32_t* row_counts, const float* y, const float* z, int32_t sectors_per_slice,
                           const tpc_track** tracks, int32_t* n_tracks, const uint32_t** cluster_ids, int64_t* n_cluster_ids);

/* ---- Track merging without any allocation (for callers that cannot call cudaMalloc: code under CUDA graph capture,
 * tight serving loops, harnesses that forbid it) ----
 * The K7 kernels of tpc_merge_tracks (same reading S7, same arithmetic, same links and chi2) with their scratch - the
 * tracks' keys, the (sector, first row) bin table, the ordered track list, the best-partner words, the counters - in
 * ONE file-scope `static __device__` array of the library instead of a tracker workspace: no tracker, no workspace,
 * and neither this call nor anything it calls uses cudaMalloc, cudaFree, cudaMallocHost or an allocating library
 * routine.  The array is sized for TPC_NO_ALLOC_MAX_TRACKS tracks and TPC_NO_ALLOC_MAX_BINS = n_sectors * n_rows bins
 * (about 1.7 MB); every GPU on which the library's kernels are loaded holds it until the process exits.
 *
 * Inputs (caller-owned DEVICE memory of the current device): dev_tracks[n_tracks] as tpc_get_tracks returns them
 * (sector < n_sectors, first_row <= last_row < n_rows, cluster_offset into dev_cluster_ids), dev_cluster_ids = the
 * cluster-id array of the same event (only the first id of each track is read: it is the track's canonical key).
 * Outputs (caller-owned DEVICE memory, n_tracks entries each): dev_next / dev_prev / dev_chi2 as tpc_get_merged's
 * next / prev / chi2.  params: host pointer or NULL = defaults; kf_smax, merge_chi2 and merge_max_row_gap are used.
 * Asynchronous on cuda_stream (a cudaStream_t of the current device, NULL = default stream): the outputs are valid
 * once the stream has reached the end of the call's work.
 *
 * The scratch is shared by every call on the same device and keeps the last call's contents; each call clears what
 * must start clean (bin counts, cursors, best-partner words, counters) on the stream before it uses it.  Calls whose
 * GPU work overlaps on one device - two streams, two host threads - RACE on the scratch: serialise them (one stream,
 * or an event between them).  The first call on a device looks the array's address up (cudaGetSymbolAddress, once
 * per device, under a lock).
 * Errors: TPC_E_ARG (null pointer with n_tracks > 0, n_tracks < 0, geometry or parameters out of their domain),
 * TPC_E_LIMIT (n_tracks > TPC_NO_ALLOC_MAX_TRACKS or n_sectors * n_rows > TPC_NO_ALLOC_MAX_BINS: nothing is launched;
 * use tpc_merge_tracks with a workspace instead), TPC_E_CUDA (*cuda_error, if not NULL, receives the cudaError_t). */
#define TPC_NO_ALLOC_MAX_TRACKS 65536
#define TPC_NO_ALLOC_MAX_BINS 16384
int tpc_merge_links_no_alloc(int32_t n_sectors, int32_t n_rows, float sector_dphi, float bz_tesla, const tpc_params* params,
                             const tpc_track* dev_tracks, int32_t n_tracks, const uint32_t* dev_cluster_ids,
                             int32_t* dev_next, int32_t* dev_prev, float* dev_chi2, void* cuda_stream, int* cuda_error);

/* Stage parity hooks (tests): copy one stage's buffers, converted to canonical (load-index) form, to host_dst.
 * Synchronous; allocates temporary device memory.  bytes must equal tpc_debug_dump_bytes(t, stage). */
size_t tpc_debug_dump_bytes(tpc_tracker* t, int stage);
int tpc_debug_dump(tpc_tracker* t, int stage, void* host_dst, size_t bytes);

/* Memory-safety check of the kernels (tests; compute-sanitizer is not available on the target pool): every buffer of
 * the workspace is followed by a 256-byte guard zone that tpc_set_workspace fills with a pattern.  Synchronises and
 * returns the number of guard zones that have been written to since (0 = no kernel wrote past the end of a buffer),
 * or a negative tpc_error. */
int tpc_debug_check_guards(tpc_tracker* t);

const char* tpc_strerror(int code);
int tpc_last_cuda_error(const tpc_tracker* t);
/* Number of kernel launches one tpc_track_sectors enqueues (for bench.py's gpu_launches). */
int tpc_launches_per_track(const tpc_tracker* t);

#ifdef __cplusplus
}
#endif
#endif /* TPCTRK_H */
