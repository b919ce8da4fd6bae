/* tpcst.h — C ABI of the B200-native TPC sector tracker (arXiv 1712.09407, "ALICE HLT TPC
 * Tracking of Pb-Pb Events on GPUs").
 *
 * The paper states the problem as: TPC clusters "are sent to the sector tracker which reconstructs
 * the tracks in each TPC sector individually"; the tracker runs a neighbours finder
 * and an evolution step (L40-L41), builds tracklets from chains of one-to-one links (L43), fits
 * and extends them with a Kalman filter (L45), selects among overlapping candidates (L46, L78,
 * L116) and "outputs a list of clusters for each track" with its fitted parameters (L102).  The
 * calls below are that statement: create a tracker for a geometry and a set of cuts, hand it the
 * clusters of one event grouped by (sector, pad row), get tracks back.
 *
 * Everything quantitative the paper leaves open (search windows, chi2 cut, state parametrisation,
 * ...) is a field of tpcst_cuts; DESIGN.md section 3 defines each one ("readings" G1..G32).
 *
 * Conventions
 *  - All functions return an int status: TPCST_OK (0) or a negative TPCST_ERR_* code.  No
 *    exceptions cross the ABI, nothing aborts, there is no CPU fallback: every step of the path
 *    runs in CUDA kernels on the device that owns `dev_workspace`.
 *  - "host" / "device" is stated for every pointer.  The caller owns every buffer it passes in;
 *    the library owns only the context and the pinned host buffers results are returned in.
 *  - Not thread-safe per context; use one context per host thread.
 */
#ifndef TPCST_H
#define TPCST_H

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#define TPCST_OK 0
#define TPCST_ERR_ARG (-1)      /* null pointer, unsorted row_start, inconsistent sizes, bad cuts (for
                                   TPCST_DEVICE input the row_start checks are made on the device and
                                   reported by the wait)                                               */
#define TPCST_ERR_RANGE (-2)    /* a (sector,row) holds more than 65535 clusters, a sector more than
                                   2^20 - 16 * (n_rows + 1) clusters, or a row's grid more than 49152
                                   bins                                                               */
#define TPCST_ERR_CAPACITY (-3) /* more clusters / tracklets / tracks than the workspace was sized for
                                   (a noisy sector must produce an error, not a hang);
                                   the event's outputs are invalid, the context stays usable           */
#define TPCST_ERR_CUDA (-4)     /* a CUDA runtime call failed; tpcst_error_string gives the text       */
#define TPCST_ERR_STATE (-5)    /* wait on a slot with nothing submitted, submit on a busy slot        */
#define TPCST_ERR_STATIC_LIMIT (-6) /* tpcst_select_owners_static: more clusters than its fixed scratch holds */

/* Where the cluster arrays of an event live. */
#define TPCST_HOST_PINNED 0
#define TPCST_HOST_PAGEABLE 1
#define TPCST_DEVICE 2

#define TPCST_N_SLOTS 4         /* events in flight (BASELINE.json configs[4])                         */

typedef struct tpcst_ctx tpcst_ctx; /* opaque */

/* Detector geometry (2 x 18 trapezoidal sectors, 159 pad rows).  Copied at create. */
typedef struct tpcst_geometry {
  uint32_t n_sectors;    /* 1..36; sectors are tracked independently (L28)                              */
  uint32_t n_rows;       /* 3..255 (159 for the TPC)                                                    */
  const float* row_x;    /* HOST [n_rows], cm, strictly increasing: local x of each pad row             */
  float tan_half_angle;  /* tan of the sector half opening angle (tan 10 deg): ymax[k] = row_x[k] * it  */
  float z_max;           /* cm; local z of clusters lies in [0, z_max] (250)                            */
  float bz_tesla;        /* solenoid field (0.5); only used to convert curvature to q/pT                */
} tpcst_geometry;

/* Every free parameter of the method.  tpcst_default_cuts fills it. */
typedef struct tpcst_cuts {
  float bin_y, bin_z;          /* G4: grid bin size in y and z, cm (1, 4).  Acceleration only.          */
  float grid_pad;              /* G4: widening of every bin lookup box, cm (1e-3)                       */
  float nf_wy_slope, nf_wy_const, nf_wz_slope, nf_wz_const; /* G6: neighbour windows                    */
  float nf_max_dev2;           /* G7: max squared straight-line deviation, cm^2 (0.25)                  */
  uint32_t min_chain_clusters; /* G12: shortest chain that seeds a tracklet (3)                         */
  float err_y2, err_z2;        /* G17: cluster variances, cm^2 (0.0144)                                 */
  float q_sinphi, q_dzds;      /* G18: process noise per row step (1e-6)                                */
  float c0_sinphi, c0_dzds, c0_kappa; /* G15: prior variances (0.25, 1.0, 2.5e-3)                       */
  float max_sinphi;            /* G16b: |sin phi| limit (0.95)                                          */
  float chi2_cut;              /* G20: pickup chi2 (2 dof) cut (10)                                     */
  uint32_t max_row_gap;        /* G21: consecutive missed rows tolerated while extrapolating (4)        */
  float edge_margin;           /* G23: cm beyond the sector edge that still counts as inside (1)        */
  uint32_t min_clusters;       /* 30                                                     */
  float min_pt;                /* L46 "cut for low momentum", GeV/c (0.05)                              */
  uint32_t select_mode;        /* 0: longest wins, first on ties (L46, L78).  1: weight
                                  n*(alpha - chi2/ndf) (L80-L94)                                        */
  float alpha;                 /* L94: chi2-suppression factor (6)                                      */
  uint32_t global_tracking;    /* PAPER.md section 5 (L116-L136): 1 = prolong track ends into the
                                  neighbouring sector (G33-G36; needs n_sectors = 18 or 36) (0) */
  uint32_t gt_max_rows;        /* G33: an end qualifies if at most this many rows lie beyond it, <= 32 (30) */
  float gt_edge;               /* G33: ... and its state lies within this distance of the sector edge, cm (3) */
  uint32_t select_rounds;      /* G26b (NEXT-4): 1 = single selection round; 2 = the clusters of tracklets that
                                  failed the cuts are released and claimed again by the accepted ones (1)  */
  uint32_t merge_tracks;       /* NEXT-3 (G37-G40): 1 = sort the sector tracks, refit
                                  them from their cluster lists and link segments across sector boundaries (0)  */
  uint32_t merge_max_gap;      /* G39: rows between the last cluster of a segment and the first of its
                                  continuation, at most (10)                                              */
  float merge_chi2_cut;        /* G39: cut on the 5-parameter match chi2 (30)                             */
  uint32_t max_passes;         /* G22d (NEXT-4, "repeated until no more clusters are found"): construction
                                  passes over a tracklet, 2..64 (2: one upward, one downward); 0 is read as the default, 2
                                  (the field is the newest one: a struct filled by hand for an older header leaves it 0;
                                  every other field must come from tpcst_default_cuts or be set).  > 2: pass 3 goes up
                                  again, pass 4 down, ... until a pass picks up nothing new.  Not combined with
                                  global_tracking (TPCST_ERR_ARG).                                          */
} tpcst_cuts;

/* Clusters of one event (L18 "ionization points ... are called clusters"), grouped by
 * (sector, row): the clusters of sector s, row k are [row_start[s*n_rows+k], row_start[s*n_rows+k+1]).
 * A cluster's identity is its index in this array; all outputs refer to it. */
typedef struct tpcst_clusters {
  const float* xyz;          /* [n_clusters*3] sector-local (x, y, z) in cm, fp32; x is not used by the
                                tracker (row_x[k] is), it is carried for the caller's convenience       */
  const uint32_t* row_start; /* [n_sectors*n_rows + 1] non-decreasing, row_start[last] == n_clusters    */
  uint32_t n_clusters;
  int32_t location;          /* TPCST_HOST_PINNED | TPCST_HOST_PAGEABLE | TPCST_DEVICE: where BOTH
                                arrays live.  Host arrays are copied on the copy stream; device arrays
                                are read in place and must stay valid until the wait returns.           */
} tpcst_clusters;

/* One sector track (L45 fitted parameters, L102 cluster list).  112 bytes. */
typedef struct tpcst_track {
  uint32_t sector;
  uint32_t first_row, last_row; /* fitted row range of the tracklet                                     */
  uint32_t n_clusters;          /* clusters kept after selection (>= min_clusters)                      */
  uint32_t first_cluster;       /* offset of this track's list in tpcst_tracks.cluster_ids              */
  uint32_t seed_cluster;        /* input index of the tracklet's start cluster                          */
  float x_ref;                  /* where the parameters are given: row_x[first_row]; with max_passes > 2,
                                   row_x[last_row] if the last pass that changed the tracklet went upwards   */
  float y, z, sinphi, dzds, qpt; /* state at x_ref; qpt = q/pT in (GeV/c)^-1                            */
  float cov[15];                /* covariance of (y, z, sinphi, dzds, kappa), lower triangle, row-major */
  float chi2;                   /* sum of chi2 increments of the final (downward) fit pass              */
} tpcst_track;

/* One prolongation of a track end into the neighbouring sector (global tracking, PAPER.md
 * section 5: "The track parameters are then converted to the coordinate system of the neighboring
 * sectors and the tracklet construction step is continued").  112 bytes. */
typedef struct tpcst_global_ext {
  uint32_t track;               /* index into tpcst_tracks.tracks                                       */
  uint32_t sector;              /* the neighbouring sector the clusters were picked up in               */
  uint32_t end;                 /* 0: inner end (prolonged towards row 0), 1: outer end                 */
  uint32_t n_clusters;          /* clusters picked up (>= 1)                                            */
  uint32_t first_cluster;       /* offset of the list in tpcst_tracks.global_cluster_ids (pickup order) */
  uint32_t row;                 /* row of the last pickup: the parameters are given at row_x[row]       */
  float x_ref;
  float y, z, sinphi, dzds, qpt; /* state in the NEIGHBOUR's frame after the last pickup                */
  float cov[15];
  float chi2;                   /* sum of the chi2 increments of the pickups                            */
} tpcst_global_ext;

/* One record per sector track, in the order of tpcst_tracks.tracks (cuts.merge_tracks = 1): what the stage
 * after the sector tracker needs.  States are (y, z, sin phi, dz/ds, kappa) with the
 * covariance as in tpcst_track; kappa = -qpt * 0.299792458e-2 * bz.  284 bytes. */
typedef struct tpcst_merge_seg {
  uint32_t rank;                /* G37: position of the track in the canonical order (sector, first_row, seed)  */
  int32_t next, prev;           /* G40: index of the track that continues this one in the neighbouring sector /
                                   that this one continues; -1 = none                                           */
  uint32_t ok;                  /* G38: 1 = both refit passes completed; else the record is zero                */
  uint32_t row_in, row_out;     /* rows of the first and the last cluster of the list                           */
  float chi2;                   /* G38: sum of the chi2 increments of the inward pass (ndf = 2 n_clusters - 5)  */
  float match_chi2;             /* G39: chi2 of the kept link to `next` (0 if none)                             */
  float in_par[5], in_cov[15];  /* state at row_x[row_in] after the inward pass                                 */
  float out_par[5], out_cov[15];/* state at row_x[row_out] after the outward pass                               */
  /* G41, the merged track: filled at the first segment of every chain (prev == -1), zero elsewhere             */
  uint32_t chain_n_seg;         /* segments of the chain through `next` (1 = not merged); 0: not a first segment,
                                   or the joint refit failed                                                    */
  uint32_t chain_n_clusters;    /* clusters of all its segments                                                 */
  float chain_chi2;             /* inward-pass chi2 of the joint refit (ndf = 2 chain_n_clusters - 5)           */
  float chain_par[5], chain_cov[15]; /* state at row_x[row_in] of this segment, in its sector's frame           */
} tpcst_merge_seg;

/* Result of one event.  Pointers are HOST (pinned, library-owned) and stay valid until the next
 * submit on the same slot or tpcst_destroy. */
typedef struct tpcst_tracks {
  uint32_t n_tracks;
  const tpcst_track* tracks;    /* in tracklet-id order = (sector, start row, start index)              */
  uint32_t n_cluster_ids;
  const uint32_t* cluster_ids;  /* input indices, per track in ascending row order                      */
  uint32_t n_tracklets;         /* tracklets constructed (before selection)                             */
  float gpu_ms;                 /* device time of the kernel set of this event (CUDA events)            */
  uint32_t n_global;            /* global tracking (cuts.global_tracking = 1), else 0:                  */
  const tpcst_global_ext* global_ext;    /* ordered by (track, end)                                     */
  uint32_t n_global_cluster_ids;
  const uint32_t* global_cluster_ids;    /* input indices                                               */
  uint32_t n_merge;             /* n_tracks if cuts.merge_tracks = 1, else 0                                    */
  const tpcst_merge_seg* merge; /* one record per track                                                         */
} tpcst_tracks;

/* Fill `cuts` with the defaults of DESIGN.md section 3. */
int tpcst_default_cuts(tpcst_cuts* cuts);

/* Bytes of device workspace tpcst_create needs for events of up to max_clusters clusters and
 * max_tracklets tracklets (all slots).  Returns 0 on bad arguments.
 * PAPER.md L142 reports what happens otherwise: "the GPU runs out of memory due to the immense amount of clusters in a noisy
 * sector" and the pipeline loses its synchronisation.  Here every buffer is sized up front from max_clusters / max_tracklets,
 * nothing is allocated per event, and an event that exceeds them comes back as TPCST_ERR_CAPACITY. */
size_t tpcst_workspace_bytes(const tpcst_geometry* geo, const tpcst_cuts* cuts, uint32_t max_clusters,
                             uint32_t max_tracklets);

/* Create a tracker ("the sector tracker which reconstructs the tracks in each TPC sector individually"; L18:
 * the geometry it is created for, 2 x 18 sectors of 159 pad rows).  dev_workspace: DEVICE memory of at least tpcst_workspace_bytes(...) bytes,
 * 256-byte aligned, owned by the caller and kept alive until tpcst_destroy.  cuda_stream_compute /
 * cuda_stream_copy: cudaStream_t handles (as void*) on the same device; the kernels of an event are ordered
 * after everything queued on the first at submit time (see tpcst_submit_event), host->device copies run on
 * the second.  *out receives the context. */
int tpcst_create(const tpcst_geometry* geo, const tpcst_cuts* cuts, uint32_t max_clusters, uint32_t max_tracklets,
                 void* dev_workspace, size_t workspace_bytes, void* cuda_stream_compute, void* cuda_stream_copy,
                 tpcst_ctx** out);

/* Track one event synchronously (submit on slot 0, then wait).  The whole path of PAPER.md L36-L46 runs between the two:
 * row grids (the "initialization" task of L52), neighbours finder (L40), evolution (L41), tracklet starts (L43), Kalman tracklet construction (L45),
 * tracklet selection (L46, L78, L116), and the output of L102: "a list of clusters for each track" plus its parameters.
 * Returns TPCST_OK, or the TPCST_ERR_* of the submit or the wait; on an error `out` is zeroed and the context stays usable. */
int tpcst_track_event(tpcst_ctx* ctx, const tpcst_clusters* clusters, tpcst_tracks* out);

/* Asynchronous form with up to TPCST_N_SLOTS events in flight, one per slot (BASELINE.json configs[4]): the
 * host->device copy of a slot's event runs on the copy stream while the kernels of the other slots' events run.
 * Every slot's kernels run on a stream of its own that the library owns, which first waits for everything queued
 * on cuda_stream_compute up to the submit (device inputs produced there are safe); the kernel sets of the events
 * in flight then overlap wherever one of them leaves SMs idle.  submit returns as soon as the work is queued
 * (TPCST_ERR_STATE if the slot still holds an event that was not waited for); wait blocks until the slot's tracks
 * are on the host.  Both calls select the context's device themselves and restore the caller's current device. */
int tpcst_submit_event(tpcst_ctx* ctx, const tpcst_clusters* clusters, int slot);
int tpcst_wait_event(tpcst_ctx* ctx, int slot, tpcst_tracks* out);

/* Intermediate results of the last event completed on `slot`, converted to the caller's index space
 * (cluster = input index) and copied to HOST memory, for stage-by-stage parity tests.
 *   what                 element type, count, meaning
 *   TPCST_DBG_BIN_OF      uint32 [N]      grid bin of each cluster inside its row (iz*ny + iy)
 *   TPCST_DBG_BIN_START   uint32 [sum over (s,k) of ny[k]*nz]  exclusive start of each bin in its row
 *   TPCST_DBG_LINKS_RAW   int32  [2*N]    up links then down links after the neighbours finder
 *   TPCST_DBG_LINKS       int32  [2*N]    the same after the evolution step
 *   TPCST_DBG_STARTS      uint32 [2*T]    start cluster of each tracklet (device result), then the length of its
 *                                         chain: the device only decides length >= min_chain_clusters, the
 *                                         accessor walks the device's evolved links on the host to report it
 *   TPCST_DBG_TRACKLETS   tpcst_track [T] every tracklet as a track record (n_clusters = nhits before
 *                                         selection, first_cluster = kept after selection)
 *   TPCST_DBG_ROW_HITS    int32  [T*R]    cluster on each row of each tracklet, or -1
 *   TPCST_DBG_OWNERS      uint32 [N]      selection key that owns each cluster (0 = none)
 *   TPCST_DBG_COUNTERS    uint32 [8]      n_clusters, n_tracklets, n_tracks, n_cluster_ids, error bits, CUDA-graph captures
 *                                         and CUDA-graph replays of this slot since tpcst_create, 0
 *   TPCST_DBG_KERNEL_MS   float  [tpcst_kernels_per_event]  device time of each kernel of the event
 *                                         (CUDA events on the compute stream; needs tpcst_set_profiling(1)
 *                                         before the submit, else TPCST_ERR_STATE)
 *   TPCST_DBG_WORK        uint64 [8]      work counters of the event: neighbour window tests, neighbour
 *                                         pair evaluations, Kalman row steps, row searches, chi2 candidates,
 *                                         updates, claimed hits, 0 (needs tpcst_set_profiling(2) before the
 *                                         submit, else TPCST_ERR_STATE).  KERNEL_MS and WORK read host-side
 *                                         state only and may be called while the other slot is in flight.
 * `cap` is the capacity of host_buf in bytes; *written receives the bytes written.  Returns
 * TPCST_ERR_ARG if cap is too small (with *written = bytes needed).  If the slot's last event ended with an error
 * (tpcst_wait_event returned TPCST_ERR_ARG / _RANGE / _CAPACITY) only TPCST_DBG_COUNTERS (with the error bits),
 * TPCST_DBG_KERNEL_MS and TPCST_DBG_WORK can be fetched; the other views return TPCST_ERR_STATE, because the
 * kernels of a failed event leave early and, for TPCST_DEVICE input, the caller's row_start did not pass validation. */
#define TPCST_DBG_BIN_OF 0
#define TPCST_DBG_BIN_START 1
#define TPCST_DBG_LINKS_RAW 2
#define TPCST_DBG_LINKS 3
#define TPCST_DBG_STARTS 4
#define TPCST_DBG_TRACKLETS 5
#define TPCST_DBG_ROW_HITS 6
#define TPCST_DBG_OWNERS 7
#define TPCST_DBG_COUNTERS 8
#define TPCST_DBG_KERNEL_MS 9
#define TPCST_DBG_WORK 10
int tpcst_debug_fetch(tpcst_ctx* ctx, int slot, int what, void* host_buf, size_t cap, size_t* written);

/* Number of kernels one event launches (for bench.py's gpu_launches), and the name of the i-th one
 * in launch order (NULL if i is out of range).  Static strings. */
int tpcst_kernels_per_event(const tpcst_ctx* ctx);
const char* tpcst_kernel_name(int i);

/* Measurement level of later submits.  0 (default): none.  1: a CUDA event is recorded on the
 * compute stream between consecutive kernels (a few microseconds per event of extra stream work);
 * TPCST_DBG_KERNEL_MS then returns the elapsed times.  2: as 1, and the kernels' counting variants
 * run, which also fill the work counters of TPCST_DBG_WORK (slower; not for timed runs).  Results
 * are identical at every level.  While profiling is on every slot's kernels run on cuda_stream_compute
 * (otherwise each slot has a stream of its own, see tpcst_submit_event), so that the times are those of
 * the kernels and not of their wait for the other event in flight. */
int tpcst_set_profiling(tpcst_ctx* ctx, int on);

/* CUDA graphs (on by default).  The kernels of an event depend on it only through the two input pointers and
 * n_clusters.  Every slot remembers the last 4 distinct triples of those values it was given (host input always gives
 * the same one: it is copied into the slot's own buffers; device input repeats when the caller reuses its buffers).
 * The second time a remembered triple comes, the slot's launch set is captured into a CUDA graph, and from then on that
 * triple is replayed with one launch; a triple that is new takes the place of the least recently used one (its graph,
 * if any, is destroyed).  Callers that alternate between up to 4 sets of buffers per slot therefore capture each once;
 * callers whose buffers never repeat never capture.  Results are identical; what changes is the host time per event.
 * on = 0 turns this off (every kernel is launched individually), on = 1 back on.  No graph is used while
 * tpcst_set_profiling is on. */
int tpcst_set_graphs(tpcst_ctx* ctx, int on);

/* Device self-test of the arithmetic helpers of construct_tracklets: the correctly rounded square
 * root and quotient written without the compiler's operand-range check are
 * compared with the IEEE operations (__fsqrt_rn, __fdiv_rn) on the current device: the square root
 * on EVERY fp32 value of [2^-8, 2^8), the quotient on n_div_pairs pseudo-random pairs with
 * |a| in [2^-24, 2^24) or a = 0 and b in [2^-8, 2^24) (the ranges the tracker produces lie far
 * inside).  cuda_stream: a cudaStream_t (as void*).  *n_checked / *n_bad (HOST pointers) receive
 * the number of comparisons and of bit-level disagreements (0 expected).  Synchronous. */
int tpcst_selftest_math(void* cuda_stream, uint64_t n_div_pairs, uint64_t* n_checked, uint64_t* n_bad);

/* Device self-test of the access pattern that bounds the selection kernels: the time the
 * current device needs for n_access 4-byte accesses at uniformly random positions of an array of n_words 32-bit words (an
 * array that fits the L2 cache for the sizes the tracker has), once as plain gathers and once as atomic maxima whose result
 * is not used.  Two small kernels with nothing of the tracker in them; each is launched twice untimed, then `reps` times
 * (1..1000), and the shortest time (CUDA events on cuda_stream) is returned in *ms_gather / *ms_red_max (HOST pointers).
 * A measured device limit to hold select_claim / select_collect against, not a step of the path.  Allocates and frees
 * its array itself.  Synchronous. */
int tpcst_selftest_random_access(void* cuda_stream, uint32_t n_words, uint64_t n_access, int reps, float* ms_gather, float* ms_red_max);

/* ---------------------------------------------------------------------------------------------
 * Tracklet selection without any allocation: tpcst_select_owners_static.
 *
 * Who this is for.  Everything else in this library works inside a workspace the caller obtains
 * from cudaMalloc (or from a framework's pool) and hands to tpcst_create.  Some callers cannot do
 * that at the point where they need the selection step: code that runs inside a real-time or
 * trigger loop where cudaMalloc's implicit device-wide synchronisation and unbounded duration are
 * not acceptable; plug-ins of a host framework that has already handed out all device memory and
 * gives a module only the buffers of its inputs and outputs; and code in a process whose memory
 * budget is fixed at start-up and audited (nothing may grow after initialisation).  For them this
 * call takes device pointers for the input and the two outputs and nothing else: the one piece of
 * scratch memory the step needs (one 32-bit claim key per cluster) is a fixed array that is part of
 * the loaded library image on every GPU.  The call itself performs no cudaMalloc, cudaFree,
 * cudaHostAlloc, stream / event creation or any other allocating runtime or library routine.
 *
 * What it computes ("the longest tracklet wins", L78 "first on ties", L116 "at least
 * 30 clusters"; G26, select_mode 0, one round): every tracklet with at least
 * `min_clusters` hits claims the clusters of its hits; a cluster goes to the claiming tracklet
 * with the most hits, and among equally long ones to the one with the lower index.  The result is
 * independent of the order in which the GPU processes the claims.  It is the same rule, with the
 * same outcome, as the select_claim / select_collect kernels of tpcst_track_event apply.
 *
 *   row_hits      DEVICE [n_tracklets][n_rows] int32: the caller's index of the cluster tracklet t
 *                 uses on row k, or -1 for "no hit on this row" (the layout of TPCST_DBG_ROW_HITS).
 *                 Any value outside [0, n_clusters) is treated as "no hit".  A tracklet's length is
 *                 the number of its hits.  Read only.
 *   n_tracklets   0 .. 2^24.       n_rows  1 .. 255.       min_clusters  1 .. 255.
 *   n_clusters    0 .. TPCST_STATIC_MAX_CLUSTERS; more returns TPCST_ERR_STATIC_LIMIT before
 *                 anything is launched.
 *   owner         DEVICE [n_clusters] uint32, written: index of the tracklet that keeps the cluster,
 *                 0xffffffff if no tracklet claims it.
 *   kept          DEVICE [n_tracklets] uint32, written: how many of its hits tracklet t keeps
 *                 (0 for a tracklet shorter than min_clusters).
 *   cuda_stream   a cudaStream_t (as void*).  The work (one memset, two kernels) is queued on it and
 *                 the call returns without waiting; outputs are valid once the stream reaches that
 *                 point.  The buffers must stay alive until then and belong to one device; the call
 *                 runs on that device whatever device is current and restores the current device.
 *
 * The fixed array.  TPCST_STATIC_MAX_CLUSTERS keys = 4 MiB of device memory, held by every GPU on
 * which this library's code has been loaded, from that moment until the process exits, whether or
 * not this call is ever made.  1 Mi clusters is one sector of a central Pb-Pb event several times
 * over, or a whole peripheral event; a whole central event (3-4 M clusters) does not fit and must
 * go through tpcst_create.
 *  - The first call on each device looks up the array's device address (cudaGetSymbolAddress) and
 *    remembers it; this may make the CUDA runtime load the library's device code onto that GPU.
 *    Make that first call during start-up, in particular before any stream capture begins.
 *  - All calls on one device share the array and it keeps the previous call's keys; every call
 *    therefore clears the part it uses before it claims.  Two calls whose work overlaps on the same
 *    GPU (different streams, or different host threads) race on it and produce garbage: keep the
 *    calls of one device on one stream, or order the streams yourself.
 * Returns TPCST_OK once the work is queued, TPCST_ERR_ARG (null pointer with a non-zero count, a
 * count or n_rows / min_clusters out of range, a buffer that is not device memory, buffers on
 * different devices), TPCST_ERR_STATIC_LIMIT, or TPCST_ERR_CUDA. */
#define TPCST_STATIC_MAX_CLUSTERS 1048576u
int tpcst_select_owners_static(const int32_t* row_hits, uint32_t n_tracklets, uint32_t n_rows, uint32_t n_clusters,
                               uint32_t min_clusters, uint32_t* owner, uint32_t* kept, void* cuda_stream);

/* Static text for a status code; for TPCST_ERR_CUDA the last CUDA error text of this thread.  (The failure PAPER.md L142
 * describes was silent; every failure of this library has a status and this text.) */
const char* tpcst_error_string(int status);

/* Waits for the context's streams, frees what the library owns (pinned result buffers, streams, events, graphs) and the
 * context; the workspace stays the caller's (the tracker is one component of a chain that outlives it).
 * Returns TPCST_ERR_ARG for a null context. */
int tpcst_destroy(tpcst_ctx* ctx);

#ifdef __cplusplus
}
#endif
#endif /* TPCST_H */
