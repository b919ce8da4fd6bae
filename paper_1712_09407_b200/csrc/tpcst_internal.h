// tpcst_internal.h — device-side data layout shared by the kernels and the host API of the CUDA
// sector tracker.  (Nothing here is used by, or uses, oracle/.)
//
// HBM layout of one event slot:
//   "sorted space": every (sector,row) owns a slab of the sorted arrays that starts at a 16-element
//   (128-byte for float2) aligned position  pstart(sr) = align16(row_start[sr] + 16*sr); the slab
//   holds the row's clusters in grid-bin order.  A cluster handle inside the pipeline is its global
//   sorted position; s_orig[] maps it back to the caller's input index.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

#include "../../include/tpcst.h"

namespace tpcst {

constexpr uint32_t kPad = 16;            // slab alignment in elements
constexpr uint32_t kMaxRowClusters = 65535;
constexpr uint32_t kMaxSectorSlabUnits = 65535;   // a sector's slabs span < 2^20 sorted positions (16 per unit)
constexpr uint32_t kMaxRowBins = 49152;  // u32 histogram must fit in shared memory (192 KB)
constexpr int kBlock = 256;              // threads per block of the per-row kernels
constexpr uint32_t kNfList = 8;          // find_neighbours: candidates per side kept in shared memory
#ifndef TPCST_KF_BLOCK
#define TPCST_KF_BLOCK 128
#endif
constexpr int kKalmanBlock = TPCST_KF_BLOCK;   // threads per block of the per-tracklet kernels
#ifndef TPCST_KF_MIN_BLOCKS
#define TPCST_KF_MIN_BLOCKS 6
#endif
constexpr int kKalmanMinBlocks = TPCST_KF_MIN_BLOCKS;   // construct_tracklets: CTAs per SM the register budget must allow

constexpr uint32_t kErrRange = 1u, kErrTrackletCap = 2u, kErrTrackCap = 4u, kErrArg = 8u;

__host__ __device__ __forceinline__ uint32_t pstart(uint32_t row_start_sr, uint32_t sr) {
  return (row_start_sr + kPad * sr + (kPad - 1u)) & ~(kPad - 1u);
}

// Per-row derived tables (DESIGN.md section 3 "Derived tables"), one 48-byte record per row.
struct __align__(16) RowTab {
  float x, ymax, ratio_up, ratio_dn;
  float w_up, w_dn, wy_up, wy_dn;
  float wz_up, wz_dn;
  uint32_t ny;        // grid columns of this row
  uint32_t bin_off;   // offset (in uint16 units) of the row's bin table inside a sector's block
};

struct Counters {
  uint32_t n_clusters, n_tracklets, n_tracks, n_ids, error;
  uint32_t kf_next;          // next tracklet id to construct (persistent construct_tracklets)
  uint32_t n_global, n_global_ids;   // global tracking: records and picked-up clusters
  // work counters, filled only by the counting variants of the kernels (tpcst_set_profiling(ctx, 2));
  // they are the units of the roofline arithmetic
  unsigned long long nf_window_tests, nf_pair_evals, kf_row_steps, kf_searches, kf_candidates, kf_updates,
      claimed_hits, pad2;
};

struct Params {
  // geometry / cuts
  uint32_t S, R, nz, bins_sector_stride;
  const RowTab* tab;
  float inv_bin_y, inv_bin_z, grid_pad, nf_max_dev2;
  float err_y2, err_z2, q_sinphi, q_dzds, c0_sinphi, c0_dzds, c0_kappa;
  float max_sinphi, chi2_cut, edge_margin, kbz, max_qpt, alpha;
  uint32_t min_chain, max_row_gap, min_clusters, select_mode;
  uint32_t max_passes;                     // NEXT-4 (G22d): construction passes, >= 2
  uint32_t select_rounds, sel_round;       // NEXT-4 (G26b): rounds asked for; round the launch belongs to (0, 1)
  uint32_t global_tracking, gt_max_rows;   // NEXT-2 (G33-G36)
  float gt_edge, gt_cos, gt_sin;
  uint32_t merge_tracks, merge_max_gap;    // NEXT-3 (G37-G40)
  float merge_chi2_cut;
  uint32_t max_clusters, npad, tcap, kcap, nf_smem_bytes, hist_smem_bytes;
  uint32_t n_clusters;       // of this event, as the caller stated it
  uint32_t hist_words;       // bin_rows: 32-bit words of its histogram (the staging area follows it in shared memory)
  uint32_t hit_stride;       // uint16 per tracklet in `hits` (R rounded up to 8)
  uint32_t kf_grid, kf_smem_bytes;   // construct_tracklets: persistent grid, dynamic shared memory
  uint32_t hit_groups, sel_grid;   // groups of 32 rows per tracklet; grid of the item-walking selection kernels
  // event input (device)
  const float* xyz;
  const uint32_t* row_start;
  // sorted space
  float2* s_yz;
  uint32_t* s_orig;
  uint16_t* bins;            // per (s,k): ny*nz + 1 exclusive starts (row-local), 16-byte aligned tables
  uint32_t* bin_of;          // [N] original index space: bin | rank_in_bin << 16
  int32_t *up_raw, *dn_raw, *up, *dn;   // links in sorted space (global sorted positions, -1 = none)
  unsigned long long* owner; // selection key per sorted position: 64-bit words with select_mode 1, the same memory as
                             // 32-bit words with select_mode 0 (the packed key of G26 has 32 bits) — see owner_* below
  // starts
  uint32_t* start_mark;      // [N] original index space: 0 or local sorted pos + 1 of a kept start
  uint32_t* start_list;      // per row slab: sorted positions of kept starts in original-index order
  uint32_t *row_cnt, *row_off;   // kept starts per (sector,row); exclusive scan = first tracklet id of the row
  uint32_t* ord_off;         // [R*S + 1] exclusive scan of row_cnt in (row, sector) order: work-list offsets
  uint4* t_desc;             // [tcap] work list of construct_tracklets: start, tracklet id, sector*R + row, 0
  // tracklets (SoA, stride tcap)
  uint16_t* hits;            // [tcap][hit_stride] row-local sorted index of the hit on each row, 0xffff = none
  uint32_t* t_rows;          // first_row | last_row << 8 | nhits << 16 | sector << 24
  uint32_t* t_seed;          // sorted position of the start cluster
  float* t_par;              // [5][tcap]
  float* t_cov;              // [9][tcap]: c00 c20 c22 c40 c42 c44 c11 c31 c33
  float* t_chi2;
  uint32_t* t_kept;          // kept clusters | accepted << 31
  uint8_t* t_grp;            // [tcap][8] kept clusters per group of 32 rows
  uint32_t* t_mask;          // [tcap][8] the kept rows of the group, one bit per row
  uint32_t* t_ci;            // first slot of the track's cluster-id list, 0xffffffff = not accepted
  uint32_t* t_ref;           // row the parameters are given at (allocated only if max_passes > 2, else it is first_row)
  uint32_t* partials;        // [2][n_blocks] per-block sums of (accepted, kept)
  // global tracking (allocated only if cuts.global_tracking)
  float* t_top;              // [14][tcap] state (5) + covariance (9) at the top hit row, end of the up pass
  uint32_t* trk_t;           // [kcap] tracklet id of every output track
  uint32_t* gt_pick;         // [2*kcap][32] clusters (input indices) picked up by prolongation (track, end)
  uint32_t* gt_n;            // [2*kcap] their number | row of the last one << 8
  float* gt_state;           // [15][2*kcap] state (5) + covariance (9) + chi2 after the last pickup
  uint32_t* gt_off;          // [2][2*kcap + 1] exclusive scans: record index, first cluster slot
  tpcst_global_ext* out_global;
  uint32_t* out_global_ids;
  // track merging (allocated only if cuts.merge_tracks)
  tpcst_merge_seg* mg_seg;   // [kcap] one record per output track
  unsigned long long* mg_best_a;   // [kcap] min over origins of (chi2 bits << 32 | rank of the origin)
  int32_t* mg_best_b;        // [kcap] best continuation of every track, -1 = none
  float* mg_chi_b;           // [kcap] its match chi2
  unsigned long long* mg_sortkey;  // [kcap] first_row << 32 | seed_cluster
  uint32_t* mg_word;         // [kcap] ok << 31 | row_in
  uint32_t* mg_sec;          // [S + 1] first track of every sector
  // output
  tpcst_track* out_tracks;
  uint32_t* out_ids;
  Counters* ctr;
};

// launchers (kernels_*.cu).  `ev` is null or an array of kKernelsPerEvent + 1 CUDA events: ev[0] is
// recorded by the caller before the first kernel, ev[i + 1] by the launcher after kernel i.
cudaError_t configure_ca(uint32_t hist_words, uint32_t nf_bytes, uint32_t* bin_rows_smem_bytes);
cudaError_t configure_kalman(int device, uint32_t n_sectors, uint32_t n_rows, uint32_t* grid, uint32_t* smem_bytes);
// `count` selects the kernel variants that also fill the work counters (not for timed runs).
void launch_ca(const Params& p, cudaStream_t st, cudaEvent_t* ev, bool count);      // kernels 0..4
void launch_kalman(const Params& p, cudaStream_t st, cudaEvent_t* ev, bool count);  // kernels 5..6
void launch_select(const Params& p, cudaStream_t st, cudaEvent_t* ev, bool count);  // kernels 7..12
void launch_global(const Params& p, cudaStream_t st, cudaEvent_t* ev);              // kernels 13..15 (global tracking only)
void launch_merge(const Params& p, cudaStream_t st, cudaEvent_t* ev);               // kernels 16..20 (track merging only)
constexpr int kKernelsPerEvent = 13, kKernelsGlobal = 3, kKernelsMerge = 5, kKernelsMax = kKernelsPerEvent + kKernelsGlobal + kKernelsMerge;
inline const char* kernel_name(int i) {
  static const char* const n[kKernelsMax] = {"bin_rows", "find_neighbours", "evolve_links", "find_starts", "scan_rows",
                                                  "list_tracklets", "construct_tracklets", "select_claim", "select_collect", "select_accept",
                                                  "scan_partials", "write_tracks", "write_ids",
                                             "gt_extend", "gt_scan", "gt_write",
                                             "merge_rank", "merge_refit", "merge_match", "merge_link", "merge_chain"};
  return i >= 0 && i < kKernelsMax ? n[i] : nullptr;
}
inline void mark(cudaEvent_t* ev, int i, cudaStream_t st) { if (ev) (void)cudaEventRecord(ev[i + 1], st); }

#ifdef __CUDACC__
// The selection key that owns a sorted position.  select_mode 0: 32-bit keys (G26), half the bytes to clear, to gather
// and to send to the L2 atomic units; select_mode 1: 64-bit (weight bits, then lower id).
__device__ __forceinline__ void owner_clear(const Params& p, uint32_t pos) {
  if (p.select_mode == 0u) reinterpret_cast<uint32_t*>(p.owner)[pos] = 0u; else p.owner[pos] = 0ull;
}
__device__ __forceinline__ unsigned long long owner_get(const Params& p, uint32_t pos) {
  if (p.select_mode == 0u) { const uint32_t k = reinterpret_cast<const uint32_t*>(p.owner)[pos]; return ((unsigned long long)k << 32) | k; }
  return p.owner[pos];
}
__device__ __forceinline__ void owner_claim(const Params& p, uint32_t pos, unsigned long long key) {
  if (p.select_mode == 0u) atomicMax(reinterpret_cast<uint32_t*>(p.owner) + pos, (uint32_t)key); else atomicMax(p.owner + pos, key);
}

// Early exit of a kernel of an event that has already failed (capacity, range or argument error of an earlier
// kernel, or of another CTA of this one).  The decision is taken per CTA, not per thread: the flag can be set by
// another CTA while this one reads it, and a CTA of which only some threads leave would go on with half-initialised
// shared memory.  Must be reached by every thread of the CTA.
__device__ __forceinline__ bool event_failed(const Params& p) { return __syncthreads_or(p.ctr->error != 0u) != 0; }

// Adds a per-thread work count to a global counter, one atomic per warp.  Must be reached by all
// 32 lanes of the warp.
__device__ __forceinline__ void count_add_warp(unsigned long long* dst, uint32_t v) {
  const uint32_t s = __reduce_add_sync(0xffffffffu, v);
  if ((threadIdx.x & 31u) == 0u && s) atomicAdd(dst, (unsigned long long)s);
}
#endif

}  // namespace tpcst
