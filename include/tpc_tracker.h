/* ===========================================================================
 * tpc_tracker.h  --  C ABI of the B200 (sm_100a) TPC sector tracker
 * ===========================================================================
 * The data-parallel hot path of the ALICE HLT TPC track finder of
 * arXiv:1712.09434 section 3 ("Cellular Automaton principle to
 * build track seeds ... Afterwards, it uses the Kalman filter for track fitting
 * and track following"; L123: cluster-wise CA phase, track-wise following phase;
 * L138: sectors processed individually and concurrently; L127: several events
 * concurrently on one GPU; L182: 159 pad rows; L213: clusters are identified by
 * their index).  The paper prints no formula: the arithmetic of every stage is
 * the numbered fp32 sequence of docs/ARITH_SPEC.md (cited below as SPEC n).
 *
 * Stages run by tpc_track_batch, one launch each for the WHOLE batch
 * (SURVEY.md section 8(a), rows a1..a8):
 *   a1 grid build (SPEC 2)           a2 neighbour finder (SPEC 3)
 *   a3 neighbour cleaner (SPEC 4)    a4 start-hit finder (SPEC 4, S1-S3)
 *   a5 tracklet constructor (SPEC 5, 6)
 *   a6 tracklet selector + a7 output compaction (SPEC 7)
 *   a8 batching: task = event * n_sectors + sector, all tasks in one call.
 *
 * Conventions
 *   - Plain C, no torch types.  Every pointer says HOST or DEVICE.
 *   - Ownership: every buffer passed in is caller-owned.  The library allocates
 *     device memory only in tpc_tracker_create (geometry tables, < 8 KB) and
 *     frees it in tpc_tracker_destroy.  Inputs are never written.
 *   - tpc_track_batch only ENQUEUES work on `cuda_stream` (a cudaStream_t cast
 *     to void*; NULL = the legacy default stream).  It never synchronises and
 *     never allocates.  Results are valid once the caller has synchronised the
 *     stream.  tpc_track_batch_host is the synchronous variant on host buffers.
 *   - Errors: 0 = ok, TPC_ERR_* < 0 otherwise, text in tpc_last_error().
 *     Data-dependent overflow (too many tracklets / tracks / hits for the
 *     capacities given) never writes out of bounds: it sets bits in header[2]
 *     and drops the items that do not fit, deterministically.
 *   - There is no CPU fallback: without a CUDA device every compute entry
 *     point fails with TPC_ERR_CUDA.
 * ===========================================================================*/
#ifndef TPC_TRACKER_H_
#define TPC_TRACKER_H_

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#define TPC_OK 0
#define TPC_ERR_ARGUMENT (-1)  /* NULL / inconsistent argument                     */
#define TPC_ERR_WORKSPACE (-2) /* workspace smaller than tpc_workspace_bytes says  */
#define TPC_ERR_CUDA (-3)      /* CUDA runtime error (no device, launch failure)   */

/* bits of header[2] (status), set on the device */
#define TPC_STATUS_TRACKLET_OVERFLOW 1u /* more tracklets than max_tracklets: the surplus was not built */
#define TPC_STATUS_TRACK_OVERFLOW 2u    /* more tracks than track_capacity: the surplus was not written */
#define TPC_STATUS_HIT_OVERFLOW 4u      /* more hits than hit_capacity: tracks that do not fit dropped  */
#define TPC_STATUS_TASK_TOO_LARGE 8u    /* a sector task holds 2^27 clusters or more: it gives no tracks */

/* Detector geometry (SPEC 1).  HOST memory; copied by tpc_tracker_create. */
typedef struct {
  int32_t n_sectors;    /* sector s = task % n_sectors; A side (z >= 0) iff 2*s < n_sectors */
  int32_t n_rows;       /* pad rows per sector (159), 3 <= n_rows <= 1024    */
  const float* row_x;   /* HOST [n_rows]: local x of every row, strictly increasing, > 0    */
  float tan_half_angle; /* row r spans |y| <= row_x[r]*tan_half_angle (+1 cm margin, T1)    */
  float z_max;          /* drift length; row z extent is [-1, z_max+1] (A) or mirrored (C)  */
} tpc_geometry;

/* Parameters (SPEC 8).  HOST memory; NULL in tpc_tracker_create = the defaults of SPEC 8. */
typedef struct {
  float sigma_y, sigma_z;           /* cluster errors [cm] (T7)                                 */
  float nf_hy, nf_hz, nf_chi2_max;  /* neighbour finder window and cut (N2, N3, N5)             */
  float grid_bin_min, grid_bin_max; /* grid bin size clamp [cm]; acceleration only (SPEC 2)     */
  float max_sinphi;                 /* transport fails beyond it (P4)                           */
  float c0_sinphi, c0_dzds, c0_qpt; /* seed covariance diagonal (K1)                            */
  float accept_k2, search_max;      /* pick-up window (H2)                                      */
  float turn_cov_scale;             /* covariance inflation at the turn-around (K4)             */
  int32_t min_seed_hits;            /* S3                                                       */
  int32_t max_row_gap;              /* K3, K5                                                   */
  int32_t min_track_hits;           /* K6, L2                                                   */
  int32_t nf_z_projection;          /* N1: 1 = project z from the origin (events); 0 = time-frame */
                                    /* mode (SPEC 11): z is known up to a shift only              */
} tpc_params;

/* Input clusters.  Arrays are DEVICE memory for tpc_track_batch and HOST
 * memory for tpc_track_batch_host.  Clusters are sorted by (task, row); the
 * index of a cluster in these arrays is its identity (gid).
 * x and charge are accepted and NOT read (the tracker uses
 * row_x[row]; R23: nothing in the method uses the charge); they may be NULL. */
typedef struct {
  const float* x;              /* [n_clusters] or NULL                                         */
  const float* y;              /* [n_clusters] local y [cm], finite                            */
  const float* z;              /* [n_clusters] z [cm], finite                                  */
  const uint16_t* charge;      /* [n_clusters] or NULL                                         */
  const uint32_t* row_offsets; /* [n_tasks*n_rows + 1], non-decreasing, [0] = 0, last = n_clusters */
  uint32_t n_clusters;         /* < 2^31                                                       */
  uint32_t n_tasks;            /* task = event*n_sectors + sector                              */
} tpc_clusters;

/* Outputs.  Arrays are DEVICE memory for tpc_track_batch and HOST memory for
 * tpc_track_batch_host.  Track t (0 <= t < header[0]) has its hits in
 * hit_cluster[track_hit_begin[t] .. + track_nhits[t]) as cluster gids in
 * ascending row order (L3).  Track order is deterministic run to run and
 * otherwise unspecified (L4).  Parameters are the state (y, z, sinphi, dz/dl,
 * q/pT) at x = track_x (the first row of the tracklet), covariance as 15
 * lower-triangular entries c00 c10 c11 c20 ... c44 (SPEC 5).
 * track_par is [5][track_capacity], track_cov is [15][track_capacity].
 * Every dbg_* pointer may be NULL; non-NULL ones are filled by extra untimed
 * kernels: links / cleaned links as gids indexed by gid (-1 = none), start
 * hits (S1) as an UNORDERED gid list, tracklets (before selection, K1-K6) in
 * tracklet order. */
typedef struct {
  uint32_t track_capacity, hit_capacity;
  uint32_t* header; /* [4]: n_tracks, n_hits, status bits, n_tracklets built.  On overflow [0],[1] hold
                       the totals that WOULD have been written; a track t < track_capacity is valid iff
                       track_hit_begin[t] + track_nhits[t] <= hit_capacity.                            */
  uint32_t* track_task;
  uint32_t* track_hit_begin;
  uint32_t* track_nhits;
  int32_t* track_ndf;
  float* track_x;
  float* track_par;
  float* track_cov;
  float* track_chi2;
  uint32_t* hit_cluster;
  int32_t *dbg_link_up, *dbg_link_dn, *dbg_clean_up, *dbg_clean_dn; /* [n_clusters] each */
  uint32_t* dbg_start_hits;   /* [n_clusters]                                             */
  uint32_t* dbg_n_start_hits; /* [1]                                                      */
  uint32_t dbg_tracklet_capacity;
  uint32_t* dbg_tracklet_start; /* [cap] gid of the start hit                             */
  uint32_t* dbg_tracklet_nhits; /* [cap]                                                  */
  int32_t* dbg_tracklet_map;    /* [cap][n_rows] gid or -1                                */
  float* dbg_tracklet_par;      /* [cap][5]                                               */
} tpc_tracks;

typedef struct tpc_tracker tpc_tracker;

/* Builds the fp32 tables T1..T8 of SPEC 1 on the host in the order written
 * there and uploads them.  geometry and params are HOST pointers (params may be
 * NULL).  bz_kgauss: solenoid field in kG (0.5 T = 5).  *out receives the handle. */
int tpc_tracker_create(const tpc_geometry* geometry, float bz_kgauss, const tpc_params* params,
                       tpc_tracker** out);
void tpc_tracker_destroy(tpc_tracker* tracker);

/* The defaults of SPEC 8 (HOST pointer out). */
void tpc_default_params(tpc_params* out);

/* Bytes of DEVICE workspace tpc_track_batch needs for inputs of at most
 * max_clusters clusters in max_tasks tasks.  max_tracklets bounds the number of
 * tracklets built (a5); 0 = the worst case max_clusters / min_seed_hits (chains
 * are vertex disjoint, S2).  The tracklet row maps dominate:
 * 4 * n_rows * max_tracklets bytes.  Pb-Pb-like events build one tracklet per
 * 30..35 clusters (config 3: 1.26 M for 40.7 M clusters), so max_clusters / 20
 * is a safe setting - 1.6 GB instead of 8 GB of workspace for config 3; more
 * tracklets than that set TPC_STATUS_TRACKLET_OVERFLOW and the surplus (the
 * last start hits in idx order) is not built. */
size_t tpc_workspace_bytes(const tpc_tracker* tracker, uint32_t max_clusters, uint32_t max_tasks,
                           uint32_t max_tracklets);

/* Runs a1..a8 on DEVICE buffers, asynchronously on cuda_stream.  workspace is
 * DEVICE memory of at least tpc_workspace_bytes(tracker, n_clusters, n_tasks,
 * max_tracklets) bytes, 256-byte aligned, contents undefined before and after.
 * The same tracker may be used from one stream at a time. */
int tpc_track_batch(tpc_tracker* tracker, const tpc_clusters* clusters, tpc_tracks* tracks, void* workspace,
                    size_t workspace_bytes, uint32_t max_tracklets, void* cuda_stream);

/* Same on HOST buffers (pinned memory recommended): copies y, z, row_offsets to
 * the device, runs a1..a8, copies the header and the used part of every
 * non-NULL output back, and synchronises.  workspace is DEVICE memory of at
 * least tpc_host_workspace_bytes(...).  dbg_* pointers must be NULL.
 * h2d_bytes / d2h_bytes (HOST, may be NULL) receive the bytes copied.
 * A batch of 2^20 clusters or more is cut into four runs of whole sector tasks
 * (at about 12, 45 and 80 % of the clusters; tasks are independent, PAPER.md
 * L138/L127) and pipelined over three streams of the tracker's own - copies
 * in, kernels, copies out - so that the copies of one run overlap the kernels
 * of another; the result is the single call's (same tracks, same order).
 * Work queued on cuda_stream before the call is waited for.  For fastest
 * copies the host buffers should be page-locked. */
size_t tpc_host_workspace_bytes(const tpc_tracker* tracker, uint32_t max_clusters, uint32_t max_tasks,
                                uint32_t max_tracklets, uint32_t track_capacity, uint32_t hit_capacity);
int tpc_track_batch_host(tpc_tracker* tracker, const tpc_clusters* clusters, tpc_tracks* tracks,
                         void* workspace, size_t workspace_bytes, uint32_t max_tracklets, void* cuda_stream,
                         uint64_t* h2d_bytes, uint64_t* d2h_bytes);

/* Pipelined variant of tpc_track_batch_host: two batches in flight (slot 0 and slot 1), each with a
 * DEVICE workspace of its own of tpc_host_workspace_bytes(...).  tpc_host_submit queues the upload of the
 * batch (HOST clusters, page-locked for overlap), the whole path and the download of the result sizes
 * on the tracker's own streams and returns at once; the host arrays of `clusters` must stay valid
 * until the slot is collected.  tpc_host_collect waits for the slot's batch, copies its tracks and hits
 * into the HOST arrays of `tracks` (capacities as given there; columns that are NULL are skipped) and
 * fills tracks->header.  With submit(k+1) issued before collect(k) the copies of one batch run under
 * the kernels of its neighbours (the gain of a GPU stage is lost when it waits for PCIe).
 * The result of a batch is tpc_track_batch's.  A slot must be collected before it is submitted again. */
int tpc_host_submit(tpc_tracker* tracker, int slot, const tpc_clusters* clusters, uint32_t track_capacity,
                    uint32_t hit_capacity, void* workspace, size_t workspace_bytes, uint32_t max_tracklets);
int tpc_host_collect(tpc_tracker* tracker, int slot, tpc_tracks* tracks, uint64_t* h2d_bytes, uint64_t* d2h_bytes);

/* Per-stage device counters of the LAST tpc_track_batch call on this tracker
 * (HOST pointer out, [TPC_N_COUNTERS] uint64; synchronises the stream given).
 * Only filled when the tracker was created with counters enabled through
 * tpc_tracker_enable_counters(tracker, 1) - counting costs atomics, so timed
 * runs leave it off. */
#define TPC_N_COUNTERS 16
/* 0 clusters, 1 grid bins, 2 start hits (S1), 3 tracklets built (S3), 4 tracklets kept (K6),
 * 5 chain hits fitted (K1, K2), 6 row searches (K3, K5), 7 candidates examined (H3),
 * 8 hits of kept tracklets, 9 row steps (transports of K2, K3, K5), 10 neighbour pairs (N4),
 * 11 unused, 12 row searches of the up pass (K3), 13 candidates examined in the up pass,
 * 14 row steps of the down pass that used a hit of the map without a search (K5), 15 unused. */
void tpc_tracker_enable_counters(tpc_tracker* tracker, int on);
int tpc_read_counters(tpc_tracker* tracker, void* cuda_stream, uint64_t* out);

/* Number of kernels one tpc_track_batch call launches (debug kernels excluded). */
int tpc_launches_per_batch(const tpc_tracker* tracker);

/* Per-stage device times.  With stage timing on, tpc_track_batch records one
 * CUDA event on cuda_stream before its first kernel and one after every stage
 * (a ring of TPC_STAGE_RING calls; recording costs no kernel and no sync).
 * tpc_read_stage_ms synchronises the stream, then writes to out_ms (HOST,
 * [TPC_N_STAGES]) the MEAN duration in milliseconds of every stage over the
 * calls recorded since timing was switched on (at most the last TPC_STAGE_RING)
 * and to n_calls (HOST, may be NULL) how many calls that was.  Stage i is
 * named tpc_stage_name(i) (static string, NULL beyond the last stage):
 * 0 grid build (a1), 1 neighbour finder (a2), 2 cleaner (a3), 3 start hits (a4),
 * 4..7 tracklet constructor (a5) as its four kernels - chain fit (K1, K2), up pass and
 * turn-around (K3, K4), refit of the rows that have a hit (K5), rest of the down pass with
 * finish (K5, K6) -, 8 ownership of shared clusters (K7, L1), 9 selector + output (a6, a7). */
#define TPC_N_STAGES 10
#define TPC_STAGE_RING 64
void tpc_tracker_enable_stage_timing(tpc_tracker* tracker, int on);
int tpc_read_stage_ms(tpc_tracker* tracker, void* cuda_stream, float* out_ms, uint32_t* n_calls);
const char* tpc_stage_name(int stage);

/* ---- sector-segment merger + final refit ------------------------------
 * PAPER.md L138 (section 3): the tracker "processes the TPC sectors individually but concurrently, and
 * merges the tracks segments afterward"; L140: a Kalman refit running on the GPU next to the tracker
 * is what the paper asks for next, because one that has to fetch the tracks over PCIe loses its gain.
 * docs/ARITH_SPEC.md section 9 defines the operation (the paper gives no procedure): the output state
 * of every sector track is taken to the row of its outermost hit, turned into the frame of the
 * neighbouring sector and compared there with the tracks that start within merge_max_row_gap rows
 * (chi2 over the five parameters, diagonal errors); mutual best choices become links (ties by the gid
 * of the first hit: order-free); every chain of linked segments - every unlinked track too - is
 * refitted in one filter pass from its outermost hit inwards, the state being turned where the chain
 * changes sector.
 *
 * tpc_merge_refit must follow the tpc_track_batch call whose tracks it merges, on the same stream,
 * with the same clusters, tracks, workspace and max_tracklets, and the workspace untouched in between:
 * it reads the cluster coordinates and the kept hits of every track from the tracker's workspace, so
 * nothing is copied and nothing leaves the device.  Asynchronous like tpc_track_batch.
 * If the tracker reported an overflow (header[2] != 0) the merger does nothing and sets
 * TPC_MERGE_STATUS_INPUT_OVERFLOW. */
typedef struct {
  float merge_chi2_max;      /* G4: match iff chi2 < this (default 50)                         */
  int32_t merge_max_row_gap; /* G2: first row of the outer segment at most this far (default 8) */
  int32_t n_slices;          /* SPEC 11: task = (frame*n_slices + slice)*n_sectors + sector; segments of the
                              * same sector in neighbouring slices are joined too (default 1: events)    */
} tpc_merge_params;
void tpc_default_merge_params(tpc_merge_params* out);

#define TPC_MERGE_STATUS_INPUT_OVERFLOW 1u /* the tracks came with an overflow status: nothing merged */
#define TPC_MERGE_STATUS_CAPACITY 2u       /* more sector tracks than `capacity`: the surplus was ignored */

/* Output of the merger.  Every pointer is DEVICE memory owned by the caller, `capacity` slots each
 * (capacity >= the number of sector tracks, e.g. tpc_tracks::track_capacity). */
typedef struct {
  uint32_t capacity;
  uint32_t* header;        /* [4]: merged tracks, links, status bits (TPC_MERGE_STATUS_*), 0          */
  int32_t* seg_next;       /* [capacity] per sector track: the track that continues it outwards, or -1 */
  int32_t* seg_prev;       /* [capacity] per sector track: the track it continues, or -1               */
  uint32_t* merged_first;  /* per merged track: its innermost sector track; merged tracks are in the   */
                           /* order of this index                                                      */
  uint32_t* merged_nseg;   /* sector tracks in the chain                                               */
  uint32_t* merged_nhits;  /* kept hits of all its segments                                            */
  uint32_t* merged_nfit;   /* hits the refit used (F3; < merged_nhits: it stopped early; 0: no refit)   */
  uint32_t* merged_sector; /* sector whose local frame the parameters are in                           */
  int32_t* merged_ndf;     /* 2 * merged_nfit - 5                                                      */
  float* merged_x;         /* x of the parameters (row of the innermost hit)                           */
  float* merged_par;       /* [5][capacity] y, z, sin(phi), dz/ds, q/pT                                */
  float* merged_cov;       /* [15][capacity] lower triangle                                            */
  float* merged_chi2;
} tpc_merged;

size_t tpc_merge_workspace_bytes(const tpc_tracker* tracker, uint32_t track_capacity, uint32_t max_tasks);
int tpc_merge_refit(tpc_tracker* tracker, const tpc_clusters* clusters, const tpc_tracks* tracks,
                    const tpc_merge_params* params, tpc_merged* merged, void* workspace, size_t workspace_bytes,
                    uint32_t max_tracklets, void* merge_workspace, size_t merge_workspace_bytes, void* cuda_stream);

/* ---- cluster transformation -------------------------------------------
 * PAPER.md L77 (footnote 1): "The TPC cluster transformation map is needed to convert the raw TPC
 * clusters from TPC pad row, TPC pad, and time coordinates into x, y, and z coordinates taking into
 * account the calibration"; L101 / L213: the map is the default or the fed-back calibration, and the
 * index of a cluster is not changed.  docs/ARITH_SPEC.md section 10 (X1..X4) defines the arithmetic
 * (the paper gives none): nominal pad/time geometry plus a bilinear (dy, dz) correction from a
 * map_ny x map_nz grid of knots per (sector,row).  The output (y, z) is what tpc_track_batch reads;
 * x is the row's (R18).  All tables are HOST memory, copied by tpc_transform_create. */
typedef struct {
  const float* pad_pitch;  /* [n_rows] width of a pad in cm                                        */
  const int32_t* n_pads;   /* [n_rows] pads of the row (>= 2)                                      */
  float t0;                /* time bin of a cluster at the end plate                               */
  float v_drift;           /* cm per time bin                                                      */
  float t_max;             /* time bin of the central electrode (> 0): the map spans [0, t_max]    */
  int32_t map_ny, map_nz;  /* knots across the pads and along the time, both >= 2                  */
  const float* map;        /* [n_sectors][n_rows][map_nz][map_ny][2] (dy, dz) in cm                */
} tpc_calibration;
typedef struct tpc_transform tpc_transform;
int tpc_transform_create(const tpc_geometry* geometry, const tpc_calibration* calibration, tpc_transform** out);
void tpc_transform_destroy(tpc_transform* transform);
/* pad, time, y, z: DEVICE [n_clusters] (16-byte aligned, e.g. from cudaMalloc), sorted by (task,row) like
 * tpc_clusters; row_offsets: DEVICE [n_tasks*n_rows + 1].  Asynchronous on cuda_stream, no allocation.
 * Returns TPC_OK or a negative code; the text is in tpc_transform_last_error. */
int tpc_transform_clusters(tpc_transform* transform, const float* pad, const float* time, const uint32_t* row_offsets,
                           uint32_t n_clusters, uint32_t n_tasks, float* y, float* z, void* cuda_stream);
const char* tpc_transform_last_error(const tpc_transform* transform);

/* ---- time frames ---------------------------------------------------------
 * continuous read-out gives "time frames with many overlapping events"; "One solution
 * is to slice the time frames along the time / beam axis, process the slices individually, and merge the
 * track segments afterwards".  docs/ARITH_SPEC.md section 11.  In a frame z is the frame coordinate zeta
 * (known up to the shift of the event), so the tracker is created with tpc_params.nf_z_projection = 0;
 * tpc_slice_frames re-sorts the clusters of whole frames - sorted by (frame, sector, row) - by
 * (frame, slice, sector, row), slice = min((int)(|zeta| / slice_len), n_slices - 1), stable inside a row;
 * tpc_track_batch then runs on n_tasks_in * n_slices tasks (any run of them per call), and
 * tpc_merge_refit with tpc_merge_params.n_slices joins the segments across sectors and slices.
 * src_index[k] = input index of output cluster k (the identity of a cluster, L213).
 * All arrays DEVICE memory; y_out, z_out, src_index: [n_clusters]; row_offsets_out:
 * [n_tasks_in*n_slices*n_rows + 1]; workspace: tpc_slice_workspace_bytes(...) bytes.  Asynchronous. */
size_t tpc_slice_workspace_bytes(uint32_t n_tasks_in, int32_t n_rows, int32_t n_slices);
int tpc_slice_frames(const float* y, const float* zeta, const uint32_t* row_offsets_in, uint32_t n_clusters,
                     uint32_t n_tasks_in, int32_t n_sectors, int32_t n_rows, float slice_len, int32_t n_slices,
                     float* y_out, float* z_out, uint32_t* src_index, uint32_t* row_offsets_out, void* workspace,
                     size_t workspace_bytes, void* cuda_stream);

/* The frame slicer for callers that cannot allocate (code under CUDA graph capture, tight serving loops,
 * harnesses that forbid cudaMalloc): the same kernels and the same result as tpc_slice_frames, but the scratch
 * (the counts of the output rows) lives in a file-scope `static __device__` array of the library instead of a
 * caller workspace.  The array holds TPC_SLICE_STATIC_MAX_ENTRIES uint32 (4 MiB; every GPU that loads the
 * library holds it until the process exits); a call needs n_tasks_in*n_rows*n_slices + 2 of them and is
 * refused with TPC_ERR_WORKSPACE (text in tpc_last_error(NULL)) beyond that - e.g. 36 sectors x 159 rows x
 * 4 slices fit 45 frames per call.  Inputs and outputs are the caller's DEVICE arrays as in tpc_slice_frames.
 * Neither call allocates or frees anything (no cudaMalloc, cudaFree or allocating library routine).
 * tpc_slice_static_setup resolves the device address of the array for the CURRENT device
 * (cudaGetSymbolAddress, once per device, not a stream operation); call it once per device at set-up, before
 * any capture - tpc_slice_frames_static does it itself on its first call on a device otherwise.
 * Every call on a device shares the one array, which keeps the last call's contents: nothing in it has to
 * start at zero (the count kernel writes every entry a call reads), but two calls that overlap on the GPU
 * (different streams, or graphs replayed side by side) race on it - keep them in stream order.
 * Asynchronous on cuda_stream. */
#define TPC_SLICE_STATIC_MAX_ENTRIES (1u << 20)
int tpc_slice_static_setup(void);
int tpc_slice_frames_static(const float* y, const float* zeta, const uint32_t* row_offsets_in, uint32_t n_clusters,
                            uint32_t n_tasks_in, int32_t n_sectors, int32_t n_rows, float slice_len, int32_t n_slices,
                            float* y_out, float* z_out, uint32_t* src_index, uint32_t* row_offsets_out,
                            void* cuda_stream);

/* ---- ITS standalone tracker -----------------------------------------------
 * PAPER.md L156-160 (section 4.2): from the clusters of the 6 ITS layers and the primary vertex, "pairs of
 * SPD clusters seen under nearly the same angle from the vertex point" seed a Kalman filter "propagated
 * outwards starting from the vertex, considered as a measured point", which attaches "the SDD and SSD
 * clusters closest to extrapolation point, provided they meet a strict track-to-cluster chi2 cut", with
 * "multiple scattering ... using average material budget per layer"; "At least 4 clusters are required per
 * track" and "tracks with 2 consecutive layers without contribution are rejected"; the outward kinematics
 * is recorded and an "inward Kalman propagation is performed to obtain the kinematics at the vertex
 * region".  docs/ARITH_SPEC.md section 12 defines every step (V1..V5, W1..W4, O1..O4, N1..N3).
 * Input: clusters of n_events events sorted by (event, layer), global x, y, z (DEVICE, fp32),
 * layer_offsets (DEVICE [n_events*6 + 1]), vertex (DEVICE [n_events][3]).  A cluster is identified by
 * its index in these arrays.  Output (DEVICE, caller-owned, `capacity` slots): per track its event, the
 * cluster of every layer or -1, the number of clusters, the frame of the track (cos, sin of the direction
 * vertex -> its layer-1 cluster; x along it, origin at the vertex), the outward state at the outermost
 * cluster and the inward state at the vertex plane, each as 22 floats x, p[5], C[15], chi2, and ndf.
 * header[4]: tracks, tracklets, status bits (1: more tracklets than the workspace holds, 2: more tracks
 * than capacity), 0.  Tracks are in the order of their layer-0 cluster.  Asynchronous on cuda_stream. */
typedef struct { float R[6], sig_rphi[6], sig_z[6], xx0[6]; } tpc_its_geometry;
typedef struct {
  float max_sinphi_pair, max_dtan; /* V3: tracklet window in sin(dphi) and in d(tan lambda)           */
  float sig_sinphi, sig_tan;       /* V4: weights of the tracklet metric                              */
  float sig_vtx_xy, sig_vtx_z;     /* W3, W4: the vertex as a measured point [cm]                     */
  float chi2_max, max_dx;          /* O2: strict track-to-cluster cut; |x_cluster - x_track| bound    */
  float c0_sinphi, c0_dzds, c0_qpt, turn_cov_scale, max_sinphi; /* as tpc_params                      */
  int32_t min_clusters;            /* O3 (4)                                                          */
} tpc_its_params;
typedef struct {
  uint32_t capacity;
  uint32_t* header;      /* [4] */
  uint32_t* event;       /* [capacity] */
  int32_t* cluster;      /* [capacity][6] */
  uint32_t* n_clusters;  /* [capacity] */
  float* frame;          /* [capacity][2] */
  float* out_state;      /* [capacity][22] */
  float* in_state;       /* [capacity][22] */
  int32_t* out_ndf;      /* [capacity] */
  int32_t* in_ndf;       /* [capacity] */
} tpc_its_tracks;
typedef struct tpc_its_tracker tpc_its_tracker;
void tpc_its_default_params(tpc_its_params* out);
int tpc_its_create(const tpc_its_geometry* geometry, float bz_kgauss, const tpc_its_params* params, tpc_its_tracker** out);
void tpc_its_destroy(tpc_its_tracker* tracker);
size_t tpc_its_workspace_bytes(const tpc_its_tracker* tracker, uint32_t max_clusters, uint32_t max_events);
int tpc_its_track_batch(tpc_its_tracker* tracker, const float* x, const float* y, const float* z,
                        const uint32_t* layer_offsets, const float* vertex, uint32_t n_clusters, uint32_t n_events,
                        tpc_its_tracks* tracks, void* workspace, size_t workspace_bytes, void* cuda_stream);
const char* tpc_its_last_error(const tpc_its_tracker* tracker);

/* Text of the last error on this tracker (never NULL). With tracker == NULL: the
 * last error of tpc_tracker_create on this thread. */
const char* tpc_last_error(const tpc_tracker* tracker);

#ifdef __cplusplus
}
#endif
#endif /* TPC_TRACKER_H_ */
