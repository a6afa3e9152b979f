/*
 * tpc_tracker.h -- C ABI of the B200-native TPC sector tracker (libtpctrk.so).
 *
 * The operation: the "sector tracker" of /root/reference/PAPER.md:25 (section 2, "Online Tracking in
 * ALICE"): for every TPC sector individually, a Cellular Automaton forms and concatenates links of
 * adjacent hits close to a straight line into track candidates of 4 to 10 hits, the track following fits
 * the candidate, extrapolates it through the sector and picks up further clusters with a simplified
 * Kalman filter, and a selection step assigns clusters to tracks dissolving ambiguities.  Only Bz is
 * respected.  The stage list and the parameterisation (y, z, sinPhi, dz/ds, q/pt) are
 * those of BASELINE.json `north_star`; every constant and formula the paper leaves open is fixed in
 * DESIGN.md ("Readings"), identically for this library and for the CPU oracle in oracle/.
 *
 * Conventions.  Units cm, Tesla, GeV/c.  A "sector instance" is one sector of one event (or drift
 * window); instance i has geometric sector i % sectors_per_event, and sectors >= sectors_per_event/2
 * are the z < 0 side.  Clusters are in the sector-local frame: x = pad-row plane, y along the pad row,
 * z along the drift.  Everything is asynchronous on the stream given by tpc_set_stream; the library
 * never allocates device memory and never synchronises inside tpc_track_sectors.
 *
 * All functions return 0 on success or a negative TPC_ERR_* code; tpc_last_error() gives the text.
 * There is no CPU fallback: without a CUDA device every call that touches the device fails with
 * TPC_ERR_CUDA.
 */
#ifndef TPC_TRACKER_H
#define TPC_TRACKER_H

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#define TPC_OK 0
#define TPC_ERR_ARG (-1)       /* NULL / negative / misaligned argument */
#define TPC_ERR_GEOMETRY (-2)  /* n_rows out of [3,255], rows not strictly increasing, or nf_bridge_rows with unequal row steps */
#define TPC_ERR_WORKSPACE (-3) /* workspace missing or smaller than tpc_workspace_bytes() */
#define TPC_ERR_CUDA (-4)      /* a CUDA runtime call failed (text in tpc_last_error) */
#define TPC_ERR_CAPACITY (-5)  /* tpc_check_counts: an output buffer was too small (results were saturated) */
#define TPC_ERR_INPUT (-6)     /* tpc_check_counts: device-side input validation failed (row too long, ...) */
#define TPC_ERR_LIMIT (-7)     /* tpc_start_hits_static: input larger than the library's built-in scratch array */

#define TPC_CAND_MAX_HITS 10   /* stride of cand_hits (reading A7: "usually 4 to 10 hits") */
#define TPC_N_COUNTS 16

typedef struct tpc_tracker tpc_tracker_t; /* opaque, library-owned */

/* Tunables.  Any field left 0 takes the default of DESIGN.md "Readings" (given in the comments). */
typedef struct {
    float nf_win_y, nf_win_z;  /* S2 neighbour window half-sizes [cm]: 2.0, 2.5 */
    float nf_d2_max;           /* S2 cut on the squared second difference [cm^2]: 1.0 */
    int32_t cand_min_hits;     /* S4 minimum chain length: 4 */
    int32_t cand_max_hits;     /* S4 hits kept per candidate: 10 (<= TPC_CAND_MAX_HITS) */
    float kf_p0[5];            /* S5 initial covariance diagonal: 1, 1, 0.1, 0.1, 10 */
    float kf_gate_sigma;       /* S5 pick-up gate in sigmas: 4 */
    float kf_win_max;          /* S5 pick-up gate cap [cm]: 3 */
    int32_t kf_max_gap;        /* S5 consecutive rows without a hit before stopping: 5 */
    float kf_max_sinphi;       /* S5 |sinPhi| limit: 0.95 */
    float kf_edge_margin;      /* S5 stop when |y| exceeds the row half-width by this [cm]: 2 */
    int32_t sel_min_hits;      /* S6 minimum hits kept by a final track: 10 */
    float grid_cell_z;         /* S1 z-bin width of the per-row grid [cm]: 6.75.  Performance only: no result depends on it */
    int32_t grid_cells_y;      /* S1 strips across a pad row (1..64): 12.  Performance only */
    int32_t nf_bridge_rows;    /* S2: 0 (default) links join adjacent pad rows only (BASELINE.json north_star);
                                  1 = a hit without an admissible adjacent pair may take one partner two rows away
                                  (single missing rows are bridged; reading A2') */
} tpc_params_t;

typedef struct {
    int32_t n_rows;            /* pad rows per sector, 3..255 (159) */
    const float* row_x;        /* HOST pointer [n_rows], strictly increasing; copied.  The steps need not be equal
                                  (reading A5': S2 weights its differences by the row steps); a step within
                                  1e-4 of the mean pitch counts as regular and keeps the default arithmetic bit for bit */
    int32_t sectors_per_event; /* 36 (even) */
    float half_angle_rad;      /* sector half opening angle (10 deg): row half-width = row_x * tan(half_angle) */
    float z_lo, z_hi;          /* z range of the z >= 0 side used for the grid (mirrored for z < 0): 0..250, or
                                  -250..500 for drift windows.  Clusters outside are legal (clamped into edge bins) */
    float sigma_y, sigma_z;    /* cluster errors used by the filter [cm] */
    tpc_params_t params;
} tpc_geometry_t;

/*
 * Output buffers: all caller-owned DEVICE memory; a NULL pointer skips that output (counts is required).
 * Index values are GLOBAL cluster indices (position in the input array) unless stated; -1 = none.
 * When a capacity is too small the library writes only what fits (never out of bounds) and `counts`
 * still holds the REQUIRED numbers, so the caller can detect it after synchronising (tpc_check_counts).
 */
typedef struct {
    /* S2/S3 (parity/debug) */
    int32_t* link_up_raw; /* [n_clusters] best up-neighbour before cleaning */
    int32_t* link_dn_raw; /* [n_clusters] */
    int32_t* link_up;     /* [n_clusters] after cleaning (mutual links only) */
    int32_t* link_dn;     /* [n_clusters] */
    /* S4 */
    int32_t* start_hits;  /* [start_capacity] ascending */
    int64_t start_capacity;
    int32_t* cand_hits;   /* [cand_capacity][TPC_CAND_MAX_HITS], unused slots -1; candidates in ascending start hit */
    int32_t* cand_n;      /* [cand_capacity] hits stored, cand_min_hits..cand_max_hits */
    int64_t cand_capacity;
    /* S5 tracklets, one slot per candidate id (parity/debug) */
    float* tl_params;     /* [tl_capacity][5] y, z, sinPhi, dz/ds, q/pt at row tl_rows[.][2] */
    float* tl_cov;        /* [tl_capacity][15] lower triangle row-major: (0,0),(1,0),(1,1),(2,0),... */
    float* tl_chi2;       /* [tl_capacity] */
    int32_t* tl_nhits;    /* [tl_capacity] attached hits; 0 = the candidate produced no tracklet */
    int32_t* tl_rows;     /* [tl_capacity][3] first row, last row, reference row */
    int32_t* tl_hits;     /* [tl_capacity][n_rows] attached cluster per row or -1 */
    int64_t tl_capacity;
    /* S6 final tracks, ascending candidate id */
    float* trk_params;    /* [trk_capacity][5] (those of the tracklet: no refit after hit removal) */
    float* trk_cov;       /* [trk_capacity][15] */
    float* trk_chi2;      /* [trk_capacity] */
    float* trk_xref;      /* [trk_capacity] x of the reference row */
    int32_t* trk_cand_id; /* [trk_capacity] */
    int32_t* trk_nhits;   /* [trk_capacity] hits kept (>= sel_min_hits) */
    int32_t* trk_sector;  /* [trk_capacity] sector instance */
    int64_t* trk_hit_offset; /* [trk_capacity+1] CSR into trk_hits */
    int32_t* trk_hits;    /* [trk_hits_capacity] kept hits, rows increasing */
    int64_t trk_capacity, trk_hits_capacity;
    int32_t* cluster_owner; /* [n_clusters] final track index or -1 */
    /* device [TPC_N_COUNTS]: 0 n_start, 1 n_cand, 2 n_tracklets, 3 n_tracks, 4 n_track_hits,
       5 input error flags (bit0: a row holds > 65535 clusters; the excess clusters are ignored),
       6 S5 transport steps executed, 7 S5 measurement updates, 8 clusters examined by the S5 pick-up search,
       9 S5 pick-up searches (work counters for the roofline arithmetic; 6-9 stay 0 unless
       tpc_set_work_counters enabled them), 10 and 13 internal, 11/12 the part of 6/7 spent on the candidates' own
       hits (fit kernel), 14-15 reserved.
       Written by the last kernel of the call. */
    int64_t* counts;
} tpc_output_t;

/* Create a tracker for one geometry and field.  Host-only work plus one small upload. */
int tpc_tracker_create(const tpc_geometry_t* geom, float bz_tesla, tpc_tracker_t** out);
void tpc_tracker_destroy(tpc_tracker_t* t);

/* Bytes of device workspace tpc_track_sectors needs for inputs up to these sizes (candidates are bounded by
   max_clusters / cand_min_hits, so no candidate count is needed). */
size_t tpc_workspace_bytes(const tpc_tracker_t* t, int64_t max_clusters, int64_t max_sector_instances);
/* The caller (PyTorch) owns the workspace; it must stay valid and unshared while a call is in flight. 256-B aligned. */
int tpc_set_workspace(tpc_tracker_t* t, void* dev_ptr, size_t bytes);
/* cudaStream_t as void*; NULL = the legacy default stream. */
int tpc_set_stream(tpc_tracker_t* t, void* cuda_stream);

/*
 * Track all sector instances (stages S1-S6).  clusters: DEVICE, 16-byte aligned, [n_clusters][4] =
 * (x, y, z, w); x and w are carried but never read (the row gives x) -- or one of the compact layouts below after
 * tpc_set_input_layout.  row_offsets: DEVICE int32
 * [n_sector_instances * n_rows + 1], CSR, instance-major row-minor, row_offsets[0] = 0 and
 * row_offsets[last] = n_clusters.  Clusters inside a row may be in any order.  n_clusters < 2^31,
 * n_sector_instances * n_rows < 2^31 - 1, and the cell tables of all rows together stay below 2^32 units of 32 bytes
 * (137 GB; n_sector_instances * n_rows * ceil((cells per row + 1) / 16) < 2^32) -- else TPC_ERR_ARG, nothing is done.
 * Asynchronous; one call in flight per tracker.
 */
int tpc_track_sectors(tpc_tracker_t* t, const void* clusters, const int32_t* row_offsets,
                      int32_t n_sector_instances, int64_t n_clusters, const tpc_output_t* out);

/*
 * Compact cluster input (PAPER.md:49 describes the experiment's own fixed-point cluster
 * formats).  x and w of a cluster are never read (the row gives x), so most of the 16 bytes per cluster are dead
 * weight on the PCIe upload (named as the bottleneck in PAPER.md:33) and in S1's read.  The layout applies to the
 * `clusters` argument of tpc_track_sectors / the host entry points and to tpc_slot_t.clusters:
 *   TPC_INPUT_XYZW  float [n][4] = (x, y, z, w), 16-byte aligned (default)
 *   TPC_INPUT_YZ    float [n][2] = (y, z), 8-byte aligned; results bit-identical to XYZW on the same (y, z)
 *   TPC_INPUT_I16   int16 [n][2] = (q_y, q_z), 4-byte aligned, 16-bit fixed point:
 *                     y = q_y * TPC_I16_Y_STEP                       (q_y signed: |y| < 128 cm, step 1/256 cm)
 *                     z = z_origin + (uint16)q_z * TPC_I16_Z_STEP    (q_z unsigned: 1024 cm range, step 1/64 cm)
 *                   with z_origin = z_lo on the z >= 0 side and -z_hi on the z < 0 side (the grid origin of that
 *                   side).  Decoding is one exact multiplication and one fp32 addition per coordinate; the tracker
 *                   then runs on the decoded fp32 (y, z) exactly as for TPC_INPUT_YZ.  Clusters outside the
 *                   representable range cannot be given in this layout: tpc_set_input_layout returns TPC_ERR_ARG
 *                   when the geometry's z range exceeds 1024 cm or the outermost row's half-width
 *                   (row_x * tan(half angle) + 0.5 cm) reaches 128 cm.
 */
#define TPC_INPUT_XYZW 0
#define TPC_INPUT_YZ 1
#define TPC_INPUT_I16 2
#define TPC_I16_Y_STEP (1.0f / 256.0f)
#define TPC_I16_Z_STEP (1.0f / 64.0f)
int tpc_set_input_layout(tpc_tracker_t* t, int32_t layout);

/* After synchronising and copying `counts` to the host: TPC_OK, TPC_ERR_CAPACITY or TPC_ERR_INPUT. */
int tpc_check_counts(const int64_t* counts_host, const tpc_output_t* out);

/* Number of kernel launches the last tpc_track_sectors call enqueued (for bench.py's gpu_launches). */
int32_t tpc_last_launch_count(const tpc_tracker_t* t);

/* Work counters of S5 (counts[6..9]): off by default.  When enabled, the follower runs a variant that also counts its
   transport steps, updates, searches and examined clusters; the results are unchanged, the call is a little slower. */
int tpc_set_work_counters(tpc_tracker_t* t, int32_t enable);

/* Optional per-stage timing: when enabled, every tpc_track_sectors call records CUDA events on its stream around
   each stage (a ring of the last TPC_TIMING_RING calls).  tpc_stage_times_ms waits for the call `age` calls back
   (0 = the last one) and returns its milliseconds in out_ms[TPC_N_STAGES]
   (order: bin, neighbours, chains, fit, follow, select; chains = S3 cleaning fused with S4, fit = the candidates'
   own hits, follow = the row-by-row extrapolation, both S5). */
#define TPC_N_STAGES 6
#define TPC_TIMING_RING 32
int tpc_set_stage_timing(tpc_tracker_t* t, int32_t enable);
int tpc_stage_times_ms(tpc_tracker_t* t, int32_t age, float* out_ms);

/*
 * Host-buffer entry points (BASELINE.json configs[4]: windows "streamed through the tracker in double-buffered
 * chunks with cluster upload overlapped on a second CUDA stream"; time frames are sliced when they do
 * not fit).  The job is cut into chunks of inst_per_chunk sector instances; chunk i+1 is uploaded while chunk i is
 * tracked and the results of earlier chunks return, each on its own stream.  A slot is the set of caller-owned DEVICE
 * buffers one chunk in flight needs (allocate 2..8).  A slot with its own workspace also gets its own compute
 * stream, so that the start of chunk i+1 overlaps the drain of chunk i's follower; slots without one share the
 * workspace given to tpc_set_workspace and a single compute stream.
 * h_clusters / h_row_offsets / the arrays of tpc_host_output_t should be pinned host memory (pageable memory works
 * but serialises the copies).  Only the arrays that are non-NULL in BOTH the slot's `out` and tpc_host_output_t are
 * produced and copied back.
 */
typedef struct {
    void* clusters;       /* device [max_clusters] records of the tracker's input layout */
    int32_t* row_offsets; /* device [max_instances * n_rows + 1] */
    int64_t max_clusters;
    int32_t max_instances;
    tpc_output_t out;     /* device outputs of this slot: counts required; trk_* / cluster_owner as wanted */
    void* workspace;      /* device, 256-B aligned, >= tpc_workspace_bytes(max_clusters, max_instances); or NULL */
    size_t workspace_bytes;
} tpc_slot_t;

typedef struct {
    /* HOST arrays for the whole job, NULL = not returned.  Indices are global: trk_hits hold positions in
       h_clusters, cluster_owner holds positions in the job-wide track list, trk_sector the job-wide instance. */
    float* trk_params;       /* [trk_capacity][5] */
    float* trk_cov;          /* [trk_capacity][15] */
    int32_t* trk_nhits;      /* [trk_capacity] */
    int32_t* trk_sector;     /* [trk_capacity] */
    int64_t* trk_hit_offset; /* [trk_capacity + 1] */
    int32_t* trk_hits;       /* [trk_hits_capacity] */
    int32_t* cluster_owner;  /* [n_clusters] */
    int64_t trk_capacity, trk_hits_capacity;
    int64_t totals[TPC_N_COUNTS]; /* written by the call: sums of the per-chunk counts */
    int64_t n_chunks, n_launches, h2d_bytes, d2h_bytes; /* written by the call */
    /* written by the call: time each stream was busy (sums of the per-chunk CUDA-event intervals; the compute
       figure can exceed wall_ms when slots have their own compute streams) and the host wall time of the call */
    float h2d_ms, compute_ms, d2h_ms, wall_ms;
} tpc_host_output_t;

/* Persistent pipeline: streams, events and the pinned counts buffer are created once, so that a run allocates
   nothing.  The slots (copied) must stay valid until tpc_pipeline_destroy; one run in flight per pipeline, and the
   tracker must not be used by other calls during a run. */
typedef struct tpc_pipeline tpc_pipeline_t;
int tpc_pipeline_create(tpc_tracker_t* t, const tpc_slot_t* slots, int32_t n_slots, tpc_pipeline_t** out);
void tpc_pipeline_destroy(tpc_pipeline_t* p);
/* Blocks until every result is on the host. */
int tpc_pipeline_run(tpc_pipeline_t* p, const void* h_clusters, const int32_t* h_row_offsets,
                     int32_t n_sector_instances, int64_t n_clusters, int32_t inst_per_chunk,
                     tpc_host_output_t* hout);

/* One-shot form: builds a pipeline on the caller's three streams (all slots share compute_stream), runs it and
   tears it down. */
int tpc_track_sectors_host(tpc_tracker_t* t, const void* h_clusters, const int32_t* h_row_offsets,
                           int32_t n_sector_instances, int64_t n_clusters, int32_t inst_per_chunk,
                           tpc_slot_t* slots, int32_t n_slots, void* h2d_stream, void* compute_stream,
                           void* d2h_stream, tpc_host_output_t* hout);

/*
 * Phase 2: sector merger + track refit ("The second phase merges the track segments found in the
 * individual sectors to final tracks and performs a track refit"; PAPER.md:33 names a GPU prototype of this fit;
 * SURVEY.md 8(f) NEXT-3).  Readings M1-M4 of DESIGN.md:
 *   refit     every final track is fitted again over the hits it KEPT in S6 (seed at the innermost kept hit, one step
 *             to the outermost, prior reset, filter inward); this replaces S6's "parameters of the tracklet, lost
 *             hits included".
 *   merge     segment B continues segment A outward iff same event/window, same z side, neighbouring sectors,
 *             first_row(B) in (last_row(A), last_row(A) + 10], and B's refitted state at its innermost hit, rotated
 *             into A's frame and transported to A's outermost row, lies within 2 cm in y and z of A's outermost hit;
 *             nearest candidate, mutual choice.
 *   merged    a chain of segments gets ONE fit: filter from the outermost hit of the outermost segment inward,
 *             rotating the state and covariance at every sector boundary; reported at the innermost hit of the
 *             innermost segment, in that segment's frame.
 * tpc_merge_refit works on the final tracks of the LAST tpc_track_sectors call of this tracker: it reads that call's
 * workspace and its row_offsets array, so it must follow it (same stream; asynchronous) before the workspace is
 * reused, and row_offsets must still be valid and unchanged.  A tpc_pipeline_run / tpc_track_sectors_host on this
 * tracker, or tpc_set_workspace with another buffer, ends that state: tpc_merge_refit then returns TPC_ERR_ARG until
 * the next tpc_track_sectors call (the pipeline's chunks live in the slots and leave nothing to merge).  Track indices
 * are those of that call (positions in trk_*).  All pointers: caller-owned DEVICE memory, NULL = skipped, counts2 required.
 */
typedef struct {
    int32_t* seg_next;   /* [n_tracks] track that continues this one outward in the neighbouring sector, or -1 */
    int32_t* seg_prev;   /* [n_tracks] the inverse link */
    int32_t* seg_ok;     /* [n_tracks] 1 = the refit of this track alone succeeded (0: |sinPhi| limit hit; keep trk_params) */
    float* seg_params;   /* [n_tracks][5] refit of the track's kept hits, at its innermost kept hit */
    float* seg_cov;      /* [n_tracks][15] */
    float* seg_chi2;     /* [n_tracks] */
    int32_t* mtrk_first; /* [mtrk_capacity] innermost segment (track index) of merged track m; ascending */
    int32_t* mtrk_nseg;  /* [mtrk_capacity] segments in the chain (1 = not merged) */
    int32_t* mtrk_nhits; /* [mtrk_capacity] kept hits of the whole chain */
    int32_t* mtrk_ok;    /* [mtrk_capacity] 1 = the chain fit succeeded */
    float* mtrk_params;  /* [mtrk_capacity][5] at the innermost hit of the innermost segment, in its sector frame */
    float* mtrk_cov;     /* [mtrk_capacity][15] */
    float* mtrk_chi2;    /* [mtrk_capacity] */
    int64_t mtrk_capacity;
    int64_t* counts2;    /* device [4]: merged tracks (required count), links, failed track refits, failed chain fits */
} tpc_phase2_output_t;

int tpc_merge_refit(tpc_tracker_t* t, const tpc_phase2_output_t* out);

/*
 * Time-coordinate tracking: vertex estimate (continuous read-out: "the tracking will run in time
 * coordinate first to estimate the vertex and only then convert to spacial coordinates").
 * In continuous read-out the z of a cluster is a drift time: the true z plus an offset common to all clusters of one
 * collision.  tpc_track_sectors and tpc_merge_refit are translation invariant in z and run on that time-like
 * coordinate unchanged; this call adds the step the paper names (readings T1-T3):
 *   T1  z_v, dca of every merged track: its closest approach to the beam line along the fitted helix
 *   T2  per event window, vertices = local maxima (3-bin sums >= 10, +-4 bins, ties to the lower bin) of the 0.5 cm
 *       histogram of z_v of the vertex-like tracks (fit ok, >= 30 hits, |dca| <= 3 cm); position = mean z_v of the
 *       vertex-like tracks within 1.5 cm of the seed bin centre; at most TPC_VTX_MAX_PER_WINDOW per window
 *   T3  every fitted track goes to the nearest vertex of its window within 3 cm, else to none; z_v of the vertex is
 *       the offset that converts the track's (and its clusters') z from the time-like to the spatial coordinate.
 * `merged` is the output struct of the preceding tpc_merge_refit call on this tracker (mtrk_first, mtrk_nhits,
 * mtrk_ok, mtrk_params and counts2 required); the call reads its arrays and the workspace, same stream, asynchronous.
 * mtrk_capacity = 0 gives an empty result (counts3 = 0, 0).  The histogram of one window sits in shared memory:
 * a geometry whose |z| range exceeds 12.7 km (200 KB of 0.5 cm bins) gets TPC_ERR_ARG here.
 */
#define TPC_VTX_MAX_PER_WINDOW 64
typedef struct {
    float* trk_zv;        /* [n_merged] z of the merged track at its closest approach to the beam line (time-like); required */
    float* trk_dca;       /* [n_merged] signed distance of closest approach in the transverse plane [cm] */
    int32_t* trk_vtx;     /* [n_merged] vertex index or -1 */
    float* vtx_z;         /* [vtx_capacity] vertices in ascending window, then ascending z */
    int32_t* vtx_window;  /* [vtx_capacity] event window (sector instance / sectors_per_event) */
    int32_t* vtx_ntracks; /* [vtx_capacity] tracks assigned to the vertex */
    int64_t vtx_capacity;
    int64_t* counts3;     /* device [2]: vertices (required count), tracks assigned to a vertex */
} tpc_vertex_output_t;

int tpc_estimate_vertices(tpc_tracker_t* t, const tpc_phase2_output_t* merged, const tpc_vertex_output_t* out);

/*
 * Start hits without any allocation (no workspace, no tracker handle).
 *
 * For callers that cannot obtain device memory: a component inside a framework that reserved the whole GPU at
 * start-up and passes each component fixed buffers only, a plug-in of an online loop where cudaMalloc is forbidden
 * because it synchronises the device under everybody else, code that was lent a stream and nothing more.  Everything
 * else in this library takes its scratch memory from the caller's workspace; this one call carries its own, a
 * file-scope __device__ array of 8 * (32 + TPC_STATIC_MAX_CLUSTERS / 2048) bytes = 512.25 KB that every GPU which
 * loads the library holds until the process exits.  The call itself runs no cudaMalloc, cudaFree or other allocating
 * routine: one cudaMemsetAsync on that array and one kernel, both on `cuda_stream` (cudaStream_t as void*, NULL = the
 * legacy default stream); asynchronous.
 *
 * The operation is the first half of S4 (link chains begin at start hits): h is a start hit iff
 * link_up[h] >= 0 and link_dn[h] < 0, where link_up / link_dn are the CLEANED links of S3 as tpc_output_t returns
 * them (index of the partner in the same arrays, -1 = none).
 *   link_up, link_dn  DEVICE int32 [n_clusters], read only (16-byte aligned arrays are read a little faster)
 *   start_hits        DEVICE int32 [start_capacity]: the start hits in ascending index; only what fits is written;
 *                     NULL allowed when start_capacity = 0 (count only)
 *   n_start           DEVICE int64 [1]: the REQUIRED count, also when it exceeds start_capacity
 * The result equals start_hits / counts[0] of tpc_track_sectors for the same links.
 *
 * Limit: n_clusters <= TPC_STATIC_MAX_CLUSTERS, else TPC_ERR_LIMIT and nothing is enqueued.  Other returns:
 * TPC_ERR_ARG (NULL / negative argument), TPC_ERR_CUDA; text from tpc_last_error(NULL) on the calling thread.
 *
 * First call on a device: it looks up the device address of the array (cudaGetSymbolAddress, once per device, with
 * the caller's current device); make that first call before starting any stream capture on that device.
 * Sharing: all calls on one device use the same array.  The call clears the part it needs, so stale contents of an
 * earlier call do no harm, but two calls that overlap on the GPU (two streams, two host threads) corrupt each other:
 * keep them on one stream or order them with events.
 */
#define TPC_STATIC_MAX_CLUSTERS (1 << 27) /* 134,217,728 */
int tpc_start_hits_static(const int32_t* link_up, const int32_t* link_dn, int64_t n_clusters, int32_t* start_hits,
                          int64_t start_capacity, int64_t* n_start, void* cuda_stream);

/* t = NULL: the text of the last failed tpc_tracker_create / tpc_start_hits_static call of the calling thread. */
const char* tpc_last_error(const tpc_tracker_t* t);

#ifdef __cplusplus
}
#endif
#endif /* TPC_TRACKER_H */
