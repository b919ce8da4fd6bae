// api.cu — host side of the C ABI declared in include/tpcst.h: derived tables, workspace carving,
// the per-event launch set (one launch set for all sectors), submit / wait with TPCST_N_SLOTS events in flight, the
// host->device copy on a side stream, and the debug accessors used by the parity tests.
#include <cmath>
#include <cstdio>
#include <cstring>
#include <new>
#include <vector>

#include "tpcst_internal.h"

using namespace tpcst;

namespace tpcst {
void launch_owners_to_orig(const Params& p, uint32_t* out, cudaStream_t st);
cudaError_t launch_selftest_math(unsigned long long n_div, unsigned long long* d_bad, cudaStream_t st);
}

namespace {

thread_local char g_cuda_err[256] = "no CUDA error recorded";

int cuda_fail(cudaError_t e, const char* what) {
  snprintf(g_cuda_err, sizeof(g_cuda_err), "%s: %s", what, cudaGetErrorString(e));
  return TPCST_ERR_CUDA;
}
#define CU(call)                                            \
  do {                                                      \
    cudaError_t e__ = (call);                               \
    if (e__ != cudaSuccess) return cuda_fail(e__, #call);   \
  } while (0)

inline size_t al(size_t v) { return (v + 255) & ~(size_t)255; }

// Every entry point that touches CUDA runs on the device that owns the workspace, whatever device is current in
// the calling thread, and leaves the caller's current device as it found it.
struct DeviceGuard {
  int prev = -1;
  cudaError_t err = cudaSuccess;
  explicit DeviceGuard(int device) {
    err = cudaGetDevice(&prev);
    if (err == cudaSuccess && prev != device) err = cudaSetDevice(device);
    else if (err == cudaSuccess) prev = -1;            // nothing to restore
  }
  ~DeviceGuard() { if (prev >= 0) (void)cudaSetDevice(prev); }
  DeviceGuard(const DeviceGuard&) = delete;
  DeviceGuard& operator=(const DeviceGuard&) = delete;
};
#define GUARD(ctx)                                                        \
  DeviceGuard guard__((ctx)->device);                                     \
  if (guard__.err != cudaSuccess) return cuda_fail(guard__.err, "select the context's device")

struct Plan {                      // sizes that depend on geometry, cuts and capacities
  uint32_t S, R, SR, nz, npad, tcap, kcap, nblk, max_clusters;
  uint32_t bins_sector_stride, max_row_bins, hit_stride;
  std::vector<RowTab> tab;
  size_t slot_bytes, shared_bytes, total_bytes;
};

struct SlotMem {                   // device pointers of one slot, carved from the workspace
  float* in_xyz; uint32_t* in_row_start;
  Params prm;
};

// The cuts as the library uses them.  max_passes was appended to tpcst_cuts in round 2: a caller that fills the struct by
// hand (or zero-initialises it) from an older header leaves it 0, which means "the default", 2.
tpcst_cuts effective_cuts(const tpcst_cuts* c) {
  tpcst_cuts e = *c;
  if (e.max_passes == 0u) e.max_passes = 2u;
  return e;
}

bool make_plan(const tpcst_geometry* g, const tpcst_cuts* c_in, uint32_t max_clusters, uint32_t max_tracklets, Plan& pl) {
  if (!g || !c_in || !g->row_x) return false;
  const tpcst_cuts eff = effective_cuts(c_in);
  const tpcst_cuts* c = &eff;
  if (g->n_sectors < 1 || g->n_sectors > 36 || g->n_rows < 3 || g->n_rows > 255) return false;
  if (!(c->bin_y > 0.f) || !(c->bin_z > 0.f) || !(g->z_max > 0.f) || !(g->tan_half_angle > 0.f)) return false;
  if (c->min_clusters < 1 || c->min_clusters > 255 || c->min_chain_clusters < 2 || !(c->min_pt > 0.f)) return false;
  if (max_clusters < 1 || max_tracklets < 1 || c->select_mode > 1 || c->select_rounds < 1 || c->select_rounds > 2) return false;
  if (c->max_passes < 2 || c->max_passes > 64 || (c->max_passes > 2 && c->global_tracking)) return false;
  if (c->merge_tracks > 1 || (c->merge_tracks && (c->merge_max_gap < 1 || !(c->merge_chi2_cut >= 0.f)))) return false;
  if (c->global_tracking > 1 || (c->global_tracking && (c->gt_max_rows < 1 || c->gt_max_rows > 32 || !(c->gt_edge >= 0.f)))) return false;
  for (uint32_t k = 0; k < g->n_rows; ++k) {
    if (!(g->row_x[k] > 0.f)) return false;
    if (k && !(g->row_x[k] > g->row_x[k - 1])) return false;
  }
  pl.S = g->n_sectors; pl.R = g->n_rows; pl.SR = pl.S * pl.R; pl.max_clusters = max_clusters;
  pl.nz = (uint32_t)std::ceil((double)g->z_max / (double)c->bin_z) + 1u;
  pl.tab.assign(pl.R, RowTab{});
  uint32_t off = 0;
  pl.max_row_bins = 0;
  for (uint32_t k = 0; k < pl.R; ++k) {           // DESIGN.md section 3 "Derived tables"
    RowTab& t = pl.tab[k];
    const double xk = (double)g->row_x[k];
    t.x = g->row_x[k];
    t.ymax = (float)(xk * (double)g->tan_half_angle);
    const double nyd = std::ceil(2.0 * (double)t.ymax / (double)c->bin_y) + 1.0;
    if (!(nyd >= 1.0) || nyd * (double)pl.nz > (double)kMaxRowBins) return false;
    t.ny = (uint32_t)nyd;
    if (k + 1 < pl.R) {
      const double xu = (double)g->row_x[k + 1];
      t.ratio_up = (float)(xu / xk);
      t.wy_up = (float)((double)c->nf_wy_slope * (xu - xk) + (double)c->nf_wy_const);
      t.wz_up = (float)((double)c->nf_wz_slope * (xu - xk) + (double)c->nf_wz_const);
    }
    if (k > 0) {
      const double xd = (double)g->row_x[k - 1];
      t.ratio_dn = (float)(xd / xk);
      t.wy_dn = (float)((double)c->nf_wy_slope * (xk - xd) + (double)c->nf_wy_const);
      t.wz_dn = (float)((double)c->nf_wz_slope * (xk - xd) + (double)c->nf_wz_const);
    }
    if (k > 0 && k + 1 < pl.R) {
      const double xu = (double)g->row_x[k + 1], xd = (double)g->row_x[k - 1];
      t.w_up = (float)((xk - xd) / (xu - xd));
      t.w_dn = (float)((xu - xk) / (xu - xd));
    }
    t.bin_off = off;
    const uint32_t nb = t.ny * pl.nz;
    pl.max_row_bins = nb > pl.max_row_bins ? nb : pl.max_row_bins;
    off += (nb + 1u + 7u) & ~7u;                  // tables start on 16-byte boundaries
  }
  pl.bins_sector_stride = off;
  pl.npad = (max_clusters + kPad * pl.SR + 2 * kPad) & ~(kPad - 1u);
  pl.tcap = max_tracklets;
  pl.nblk = (pl.tcap + kKalmanBlock - 1) / kKalmanBlock;
  const uint32_t by_len = max_clusters / c->min_clusters + 1u;
  pl.kcap = by_len < pl.tcap ? by_len : pl.tcap;
  size_t b = 0;
  b += al((size_t)max_clusters * 12) + al((size_t)(pl.SR + 1) * 4);                       // inputs
  b += al((size_t)pl.npad * 8) + al((size_t)pl.npad * 4);                                  // s_yz, s_orig
  b += al((size_t)pl.S * pl.bins_sector_stride * 2) + al((size_t)max_clusters * 4);        // bins, bin_of
  b += 4 * al((size_t)pl.npad * 4) + al((size_t)pl.npad * 8);                              // links, owner
  b += al((size_t)max_clusters * 4) + al((size_t)pl.npad * 4);                             // start_mark, start_list
  b += al((size_t)pl.SR * 4) + 2 * al((size_t)(pl.SR + 1) * 4);                            // row_cnt, row_off, ord_off
  b += al((size_t)pl.tcap * 16);                                                           // t_desc
  pl.hit_stride = (pl.R + 7u) & ~7u;               // uint16 per tracklet row of `hits` (16-byte multiple)
  b += al((size_t)pl.tcap * pl.hit_stride * 2);                                            // hits
  b += 5 * al((size_t)pl.tcap * 4) + al((size_t)pl.tcap * 20) + al((size_t)pl.tcap * 36) + al((size_t)pl.tcap * 8) + al((size_t)pl.tcap * 32);  // tracklet SoA
  b += al((size_t)pl.nblk * 8);                                                            // partials
  b += al((size_t)pl.kcap * sizeof(tpcst_track)) + al((size_t)max_clusters * 4);           // outputs
  b += al(sizeof(Counters));
  if (c->global_tracking) {                        // NEXT-2 scratch and outputs
    b += al((size_t)pl.tcap * 56) + al((size_t)pl.kcap * 4) + al((size_t)pl.kcap * 2 * 32 * 4) + al((size_t)pl.kcap * 2 * 4);
    b += al((size_t)pl.kcap * 2 * 60) + al(((size_t)pl.kcap * 2 + 1) * 8);
    b += al((size_t)pl.kcap * 2 * sizeof(tpcst_global_ext)) + al((size_t)pl.kcap * 2 * 32 * 4);
  }
  if (c->max_passes > 2) b += al((size_t)pl.tcap * 4);                                     // t_ref
  if (c->merge_tracks)                             // NEXT-3 records and scratch
    b += al((size_t)pl.kcap * sizeof(tpcst_merge_seg)) + 2 * al((size_t)pl.kcap * 8) + 3 * al((size_t)pl.kcap * 4) + al((size_t)(pl.S + 1) * 4);
  pl.slot_bytes = b;
  pl.shared_bytes = al((size_t)pl.R * sizeof(RowTab)) + al((size_t)max_clusters * 4);      // tables, debug scratch
  pl.total_bytes = pl.shared_bytes + TPCST_N_SLOTS * pl.slot_bytes;
  return true;
}

struct Slot {
  SlotMem m;
  tpcst_track* h_tracks = nullptr;
  uint32_t* h_ids = nullptr;
  tpcst_global_ext* h_global = nullptr;
  uint32_t* h_global_ids = nullptr;
  tpcst_merge_seg* h_merge = nullptr;
  Counters* h_ctr = nullptr;
  cudaEvent_t ev_h2d = nullptr, ev_start = nullptr, ev_done = nullptr, ev_ctr = nullptr;
  cudaEvent_t ev_k[kKernelsMax + 1] = {};
  bool busy = false, done = false, profiled = false, counted = false;
  bool failed = false;     // the last waited event ended with an error: its intermediate arrays (and, for device input, the
                           // caller's row_start) are not to be trusted by tpcst_debug_fetch
  // The launch set of this slot as CUDA graphs.  A graph is valid for one (xyz, row_start, n_clusters) of Params; the
  // slot remembers the last kGraphKeys distinct triples it was given.  A triple is captured the second time it comes
  // while remembered and replayed from then on; a new triple takes the place of the least recently used one.  So a
  // caller that alternates between a few input buffers (A,A,B,B or A,B,A,B) captures each once, and a caller whose
  // buffers never repeat (or cycle through more than kGraphKeys of them) never pays for a capture.
  struct GraphKey {
    const void *xyz = nullptr, *rs = nullptr;
    uint32_t n = 0, seen = 0;           // seen: submits with this triple since it entered the table
    unsigned long long used = 0;        // value of `tick` at its last submit (least recently used = smallest)
    cudaGraphExec_t graph = nullptr;
  };
  static constexpr int kGraphKeys = 4;
  GraphKey gkey[kGraphKeys];
  unsigned long long tick = 0;
  uint32_t n_captures = 0, n_replays = 0;   // since tpcst_create (TPCST_DBG_COUNTERS [5], [6])
  uint32_t n_clusters = 0;
  const uint32_t* host_row_start = nullptr;   // only valid for host-located input, for debug_fetch
  std::vector<uint32_t> row_start_copy;
};

}  // namespace

namespace tpcst {
// for the entry points that live in other files (static_select.cu): record the CUDA error text for tpcst_error_string
int cuda_status(cudaError_t e, const char* what) { return cuda_fail(e, what); }
}

struct tpcst_ctx {
  Plan plan;
  tpcst_cuts cuts;
  tpcst_geometry geo;
  float kbz;
  cudaStream_t st_compute, st_copy, st_d2h;
  cudaStream_t st_slot[TPCST_N_SLOTS] = {};   // compute stream of every slot, library-owned
  cudaEvent_t ev_dep[TPCST_N_SLOTS] = {};     // "everything the caller queued on st_compute before this submit"
  Slot slot[TPCST_N_SLOTS];
  uint32_t* d_dbg;     // [max_clusters] scratch for debug conversions
  int device;
  int profiling = 0;   // 0 off, 1 per-kernel events, 2 events + work counters
  int graphs = 1;      // replay the launch set as a CUDA graph when the same input buffers come again
};

extern "C" {

int tpcst_default_cuts(tpcst_cuts* c) {
  if (!c) return TPCST_ERR_ARG;
  c->bin_y = 1.0f; c->bin_z = 4.0f; c->grid_pad = 1e-3f;
  c->nf_wy_slope = 1.0f; c->nf_wy_const = 0.5f; c->nf_wz_slope = 0.5f; c->nf_wz_const = 0.5f;
  c->nf_max_dev2 = 0.25f;
  c->min_chain_clusters = 3;
  c->err_y2 = 0.0144f; c->err_z2 = 0.0144f;
  c->q_sinphi = 1e-6f; c->q_dzds = 1e-6f;
  c->c0_sinphi = 0.25f; c->c0_dzds = 1.0f; c->c0_kappa = 2.5e-3f;
  c->max_sinphi = 0.95f;
  c->chi2_cut = 10.0f;
  c->max_row_gap = 4;
  c->edge_margin = 1.0f;
  c->min_clusters = 30;
  c->min_pt = 0.05f;
  c->select_mode = 0;
  c->alpha = 6.0f;
  c->global_tracking = 0; c->gt_max_rows = 30; c->gt_edge = 3.0f;
  c->select_rounds = 1;
  c->merge_tracks = 0; c->merge_max_gap = 10; c->merge_chi2_cut = 30.0f;
  c->max_passes = 2;
  return TPCST_OK;
}

size_t tpcst_workspace_bytes(const tpcst_geometry* g, const tpcst_cuts* c, uint32_t max_clusters, uint32_t max_tracklets) {
  Plan pl;
  if (!make_plan(g, c, max_clusters, max_tracklets, pl)) return 0;
  return pl.total_bytes;
}

int tpcst_create(const tpcst_geometry* g, const tpcst_cuts* c, uint32_t max_clusters, uint32_t max_tracklets,
                 void* ws, size_t ws_bytes, void* s_compute, void* s_copy, tpcst_ctx** out) {
  if (!out) return TPCST_ERR_ARG;
  *out = nullptr;
  tpcst_ctx* ctx = new (std::nothrow) tpcst_ctx();
  if (!ctx) return TPCST_ERR_ARG;
  Plan& pl = ctx->plan;
  if (!make_plan(g, c, max_clusters, max_tracklets, pl)) {
    const bool range = g && c && g->row_x && c->bin_y > 0.f && c->bin_z > 0.f;
    delete ctx;
    // distinguish "grid too fine" from plain bad arguments
    if (range) {
      const double nz = std::ceil((double)g->z_max / (double)c->bin_z) + 1.0;
      const double ny = std::ceil(2.0 * (double)g->row_x[g->n_rows ? g->n_rows - 1 : 0] * (double)g->tan_half_angle / (double)c->bin_y) + 1.0;
      if (ny * nz > (double)kMaxRowBins) return TPCST_ERR_RANGE;
    }
    return TPCST_ERR_ARG;
  }
  if (!ws || ws_bytes < pl.total_bytes || ((uintptr_t)ws & 255u)) { delete ctx; return TPCST_ERR_ARG; }
  const tpcst_cuts eff = effective_cuts(c);          // make_plan succeeded: c is not null
  c = &eff;
  ctx->cuts = eff;
  ctx->geo = *g;
  ctx->geo.row_x = nullptr;
  ctx->kbz = (float)(0.299792458e-2 * (double)g->bz_tesla);
  ctx->st_compute = (cudaStream_t)s_compute;
  ctx->st_copy = (cudaStream_t)s_copy;
  cudaPointerAttributes attr;
  cudaError_t e = cudaPointerGetAttributes(&attr, ws);
  if (e != cudaSuccess || attr.type != cudaMemoryTypeDevice) { delete ctx; (void)cudaGetLastError(); return TPCST_ERR_ARG; }
  ctx->device = attr.device;
  DeviceGuard guard(ctx->device);
  if (guard.err != cudaSuccess) { delete ctx; return cuda_fail(guard.err, "select the workspace's device"); }
  if ((e = cudaStreamCreateWithFlags(&ctx->st_d2h, cudaStreamNonBlocking)) != cudaSuccess) { delete ctx; return cuda_fail(e, "cudaStreamCreate"); }

  // carve the workspace
  unsigned char* base = (unsigned char*)ws;
  size_t o = 0;
  auto take = [&](size_t bytes) { void* p = base + o; o += al(bytes); return p; };
  RowTab* d_tab = (RowTab*)take((size_t)pl.R * sizeof(RowTab));
  ctx->d_dbg = (uint32_t*)take((size_t)max_clusters * 4);
  const uint32_t hist_words = (pl.max_row_bins + 1u + 7u) & ~7u;   // counts of a row + the end marker, in whole 8-entry groups
  uint32_t hist_bytes = 0;                         // bin_rows' dynamic shared memory: histogram + staging area (configure_ca)
  uint32_t nf_bytes = 40u * 1024u;                 // + 8 KB of candidate lists: 4 CTAs/SM; larger rows read in place
  for (int s = 0; s < TPCST_N_SLOTS; ++s) {
    Slot& sl = ctx->slot[s];
    Params& p = sl.m.prm;
    std::memset(&p, 0, sizeof(p));
    sl.m.in_xyz = (float*)take((size_t)max_clusters * 12);
    sl.m.in_row_start = (uint32_t*)take((size_t)(pl.SR + 1) * 4);
    p.s_yz = (float2*)take((size_t)pl.npad * 8);
    p.s_orig = (uint32_t*)take((size_t)pl.npad * 4);
    p.bins = (uint16_t*)take((size_t)pl.S * pl.bins_sector_stride * 2);
    p.bin_of = (uint32_t*)take((size_t)max_clusters * 4);
    p.up_raw = (int32_t*)take((size_t)pl.npad * 4);
    p.dn_raw = (int32_t*)take((size_t)pl.npad * 4);
    p.up = (int32_t*)take((size_t)pl.npad * 4);
    p.dn = (int32_t*)take((size_t)pl.npad * 4);
    p.owner = (unsigned long long*)take((size_t)pl.npad * 8);
    p.start_mark = (uint32_t*)take((size_t)max_clusters * 4);
    p.start_list = (uint32_t*)take((size_t)pl.npad * 4);
    p.row_cnt = (uint32_t*)take((size_t)pl.SR * 4);
    p.row_off = (uint32_t*)take((size_t)(pl.SR + 1) * 4);
    p.ord_off = (uint32_t*)take((size_t)(pl.SR + 1) * 4);
    p.t_desc = (uint4*)take((size_t)pl.tcap * 16);
    p.hits = (uint16_t*)take((size_t)pl.tcap * pl.hit_stride * 2);
    p.t_rows = (uint32_t*)take((size_t)pl.tcap * 4);
    p.t_seed = (uint32_t*)take((size_t)pl.tcap * 4);
    p.t_chi2 = (float*)take((size_t)pl.tcap * 4);
    p.t_kept = (uint32_t*)take((size_t)pl.tcap * 4);
    p.t_ci = (uint32_t*)take((size_t)pl.tcap * 4);
    p.t_grp = (uint8_t*)take((size_t)pl.tcap * 8);
    p.t_mask = (uint32_t*)take((size_t)pl.tcap * 32);
    p.t_par = (float*)take((size_t)pl.tcap * 20);
    p.t_cov = (float*)take((size_t)pl.tcap * 36);
    p.partials = (uint32_t*)take((size_t)pl.nblk * 8);
    p.out_tracks = (tpcst_track*)take((size_t)pl.kcap * sizeof(tpcst_track));
    p.out_ids = (uint32_t*)take((size_t)max_clusters * 4);
    p.ctr = (Counters*)take(sizeof(Counters));
    if (c->global_tracking) {
      p.t_top = (float*)take((size_t)pl.tcap * 56);
      p.trk_t = (uint32_t*)take((size_t)pl.kcap * 4);
      p.gt_pick = (uint32_t*)take((size_t)pl.kcap * 2 * 32 * 4);
      p.gt_n = (uint32_t*)take((size_t)pl.kcap * 2 * 4);
      p.gt_state = (float*)take((size_t)pl.kcap * 2 * 60);
      p.gt_off = (uint32_t*)take(((size_t)pl.kcap * 2 + 1) * 8);
      p.out_global = (tpcst_global_ext*)take((size_t)pl.kcap * 2 * sizeof(tpcst_global_ext));
      p.out_global_ids = (uint32_t*)take((size_t)pl.kcap * 2 * 32 * 4);
    }
    if (c->max_passes > 2) p.t_ref = (uint32_t*)take((size_t)pl.tcap * 4);
    if (c->merge_tracks) {
      p.mg_seg = (tpcst_merge_seg*)take((size_t)pl.kcap * sizeof(tpcst_merge_seg));
      p.mg_best_a = (unsigned long long*)take((size_t)pl.kcap * 8);
      p.mg_best_b = (int32_t*)take((size_t)pl.kcap * 4);
      p.mg_chi_b = (float*)take((size_t)pl.kcap * 4);
      p.mg_sortkey = (unsigned long long*)take((size_t)pl.kcap * 8);
      p.mg_word = (uint32_t*)take((size_t)pl.kcap * 4);
      p.mg_sec = (uint32_t*)take((size_t)(pl.S + 1) * 4);
    }
    p.S = pl.S; p.R = pl.R; p.nz = pl.nz; p.bins_sector_stride = pl.bins_sector_stride; p.tab = d_tab;
    p.inv_bin_y = (float)(1.0 / (double)c->bin_y); p.inv_bin_z = (float)(1.0 / (double)c->bin_z);
    p.grid_pad = c->grid_pad; p.nf_max_dev2 = c->nf_max_dev2;
    p.err_y2 = c->err_y2; p.err_z2 = c->err_z2; p.q_sinphi = c->q_sinphi; p.q_dzds = c->q_dzds;
    p.c0_sinphi = c->c0_sinphi; p.c0_dzds = c->c0_dzds; p.c0_kappa = c->c0_kappa;
    p.max_sinphi = c->max_sinphi; p.chi2_cut = c->chi2_cut; p.edge_margin = c->edge_margin;
    p.kbz = ctx->kbz; p.max_qpt = (float)(1.0 / (double)c->min_pt); p.alpha = c->alpha;
    p.min_chain = c->min_chain_clusters; p.max_row_gap = c->max_row_gap; p.min_clusters = c->min_clusters;
    p.select_mode = c->select_mode;
    p.select_rounds = c->select_rounds; p.sel_round = 0; p.max_passes = c->max_passes;
    p.global_tracking = c->global_tracking; p.gt_max_rows = c->gt_max_rows; p.gt_edge = c->gt_edge;
    p.merge_tracks = c->merge_tracks; p.merge_max_gap = c->merge_max_gap; p.merge_chi2_cut = c->merge_chi2_cut;
    {
      const double dphi = 2.0 * std::atan((double)g->tan_half_angle);   // G34: angle between neighbouring sectors
      p.gt_cos = (float)std::cos(dphi); p.gt_sin = (float)std::sin(dphi);
    }
    p.max_clusters = max_clusters; p.npad = pl.npad; p.tcap = pl.tcap; p.kcap = pl.kcap;
    p.nf_smem_bytes = nf_bytes; p.hist_words = hist_words;
    p.hit_stride = pl.hit_stride; p.hit_groups = (pl.R + 31u) / 32u;
    if ((e = cudaHostAlloc((void**)&sl.h_tracks, (size_t)pl.kcap * sizeof(tpcst_track), cudaHostAllocDefault)) != cudaSuccess ||
        (e = cudaHostAlloc((void**)&sl.h_ids, (size_t)max_clusters * 4, cudaHostAllocDefault)) != cudaSuccess ||
        (e = cudaHostAlloc((void**)&sl.h_ctr, sizeof(Counters), cudaHostAllocDefault)) != cudaSuccess ||
        (c->global_tracking && ((e = cudaHostAlloc((void**)&sl.h_global, (size_t)pl.kcap * 2 * sizeof(tpcst_global_ext), cudaHostAllocDefault)) != cudaSuccess ||
                                (e = cudaHostAlloc((void**)&sl.h_global_ids, (size_t)pl.kcap * 2 * 32 * 4, cudaHostAllocDefault)) != cudaSuccess)) ||
        (c->merge_tracks && (e = cudaHostAlloc((void**)&sl.h_merge, (size_t)pl.kcap * sizeof(tpcst_merge_seg), cudaHostAllocDefault)) != cudaSuccess) ||
        (e = cudaEventCreateWithFlags(&sl.ev_h2d, cudaEventDisableTiming)) != cudaSuccess ||
        (e = cudaEventCreateWithFlags(&sl.ev_ctr, cudaEventDisableTiming)) != cudaSuccess ||
        (e = cudaEventCreate(&sl.ev_start)) != cudaSuccess || (e = cudaEventCreate(&sl.ev_done)) != cudaSuccess) {
      tpcst_destroy(ctx);
      return cuda_fail(e, "host buffers / events");
    }
    for (cudaEvent_t& ek : sl.ev_k)
      if ((e = cudaEventCreate(&ek)) != cudaSuccess) { tpcst_destroy(ctx); return cuda_fail(e, "cudaEventCreate"); }
  }
  if (o > ws_bytes) { tpcst_destroy(ctx); return TPCST_ERR_ARG; }
  if ((e = cudaMemcpyAsync(d_tab, pl.tab.data(), (size_t)pl.R * sizeof(RowTab), cudaMemcpyHostToDevice, ctx->st_compute)) != cudaSuccess ||
      (e = cudaStreamSynchronize(ctx->st_compute)) != cudaSuccess || (e = configure_ca(hist_words, nf_bytes, &hist_bytes)) != cudaSuccess) {
    tpcst_destroy(ctx);
    return cuda_fail(e, "table upload / kernel attributes");
  }
  uint32_t kf_grid = 0, kf_smem = 0;
  if ((e = configure_kalman(ctx->device, pl.S, pl.R, &kf_grid, &kf_smem)) != cudaSuccess) {
    tpcst_destroy(ctx);
    return cuda_fail(e, "construct_tracklets attributes");
  }
  int sms = 0;
  (void)cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, ctx->device);
  // Every slot has its own compute stream, so that the kernel sets of the events in flight overlap where one
  // of them leaves SMs idle (the drain of a persistent kernel, the tails of the per-row kernels).  The streams are
  // the library's; every submit orders its slot's stream after what the caller has queued on cuda_stream_compute
  // (which never holds the library's own kernels, so the slots do not wait for each other).
  for (int i = 0; i < TPCST_N_SLOTS; ++i) {
    if ((e = cudaStreamCreateWithFlags(&ctx->st_slot[i], cudaStreamNonBlocking)) != cudaSuccess ||
        (e = cudaEventCreateWithFlags(&ctx->ev_dep[i], cudaEventDisableTiming)) != cudaSuccess) {
      tpcst_destroy(ctx);
      return cuda_fail(e, "slot streams");
    }
  }
  for (Slot& sl : ctx->slot) { sl.m.prm.hist_smem_bytes = hist_bytes; sl.m.prm.kf_grid = kf_grid; sl.m.prm.kf_smem_bytes = kf_smem; sl.m.prm.sel_grid = (uint32_t)(sms > 0 ? sms : 148) * 8u; }
  *out = ctx;
  return TPCST_OK;
}

int tpcst_submit_event(tpcst_ctx* ctx, const tpcst_clusters* cl, int s) {
  if (!ctx || !cl || s < 0 || s >= TPCST_N_SLOTS || !cl->row_start || (cl->n_clusters && !cl->xyz)) return TPCST_ERR_ARG;
  if (cl->location < TPCST_HOST_PINNED || cl->location > TPCST_DEVICE) return TPCST_ERR_ARG;
  Slot& sl = ctx->slot[s];
  if (sl.busy) return TPCST_ERR_STATE;
  const Plan& pl = ctx->plan;
  if (cl->n_clusters > pl.max_clusters) return TPCST_ERR_CAPACITY;
  GUARD(ctx);
  Params& p = sl.m.prm;
  sl.n_clusters = cl->n_clusters;
  p.n_clusters = cl->n_clusters;                     // device row_start is checked against it by bin_rows
  sl.done = false;
  // with per-kernel profiling on, every slot runs on the caller's stream: an event pair around a kernel would
  // otherwise also time its wait for the SMs the other slot's kernels hold
  cudaStream_t st = ctx->profiling ? ctx->st_compute : ctx->st_slot[s];
  if (st != ctx->st_compute) {                       // device inputs may have been produced on the caller's stream
    CU(cudaEventRecord(ctx->ev_dep[s], ctx->st_compute));
    CU(cudaStreamWaitEvent(st, ctx->ev_dep[s], 0));
  }
  if (cl->location != TPCST_DEVICE) {
    const uint32_t* rs = cl->row_start;
    if (rs[0] != 0u || rs[pl.SR] != cl->n_clusters) return TPCST_ERR_ARG;
    for (uint32_t i = 0; i < pl.SR; ++i) {
      if (rs[i] > rs[i + 1]) return TPCST_ERR_ARG;
      if (rs[i + 1] - rs[i] > kMaxRowClusters) return TPCST_ERR_RANGE;
    }
    if (cl->n_clusters)
      CU(cudaMemcpyAsync(sl.m.in_xyz, cl->xyz, (size_t)cl->n_clusters * 12, cudaMemcpyHostToDevice, ctx->st_copy));
    CU(cudaMemcpyAsync(sl.m.in_row_start, rs, (size_t)(pl.SR + 1) * 4, cudaMemcpyHostToDevice, ctx->st_copy));
    CU(cudaEventRecord(sl.ev_h2d, ctx->st_copy));
    CU(cudaStreamWaitEvent(st, sl.ev_h2d, 0));
    p.xyz = sl.m.in_xyz; p.row_start = sl.m.in_row_start;
    p.n_clusters = 0xffffffffu;                      // validated above: bin_rows skips its row_start checks
  } else {
    p.xyz = cl->xyz; p.row_start = cl->row_start;
  }
  CU(cudaEventRecord(sl.ev_start, st));
  cudaEvent_t* ev = ctx->profiling ? sl.ev_k : nullptr;
  sl.profiled = ctx->profiling;
  const bool count = ctx->profiling >= 2;
  sl.counted = count;
  // The launch set (one memset + 13..21 kernels) depends on the event only through three fields of Params: the two
  // input pointers and n_clusters.  Host input always lands in the slot's own buffers, so its Params never change;
  // device input repeats when the caller reuses its buffers.  See Slot::GraphKey for when a triple is captured; once it
  // is, one cudaGraphLaunch replaces the individual launches (what this saves is host time per event: it shows in the
  // latency of a single small event, not in the pipelined throughput).
  const bool use_graph = ctx->graphs && !ctx->profiling;
  Slot::GraphKey* gk = nullptr;
  if (use_graph) {
    ++sl.tick;
    for (Slot::GraphKey& k : sl.gkey)
      if (k.seen && k.xyz == p.xyz && k.rs == p.row_start && k.n == p.n_clusters) gk = &k;
    if (!gk) {                                         // new triple: take a free entry, else the least recently used
      gk = &sl.gkey[0];
      for (Slot::GraphKey& k : sl.gkey) if (k.used < gk->used) gk = &k;
      if (gk->graph) (void)cudaGraphExecDestroy(gk->graph);
      *gk = Slot::GraphKey{};
      gk->xyz = p.xyz; gk->rs = p.row_start; gk->n = p.n_clusters;
    }
    ++gk->seen;
    gk->used = sl.tick;
  }
  if (gk && gk->graph) {
    CU(cudaGraphLaunch(gk->graph, st));
    ++sl.n_replays;
  } else {
    const bool capture = gk && gk->seen >= 2u;
    if (capture) CU(cudaStreamBeginCapture(st, cudaStreamCaptureModeThreadLocal));
    cudaError_t le = cudaMemsetAsync(p.ctr, 0, sizeof(Counters), st);
    if (ev && le == cudaSuccess) le = cudaEventRecord(ev[0], st);
    launch_ca(p, st, ev, count);
    launch_kalman(p, st, ev, count);
    launch_select(p, st, ev, count);
    if (p.global_tracking) launch_global(p, st, ev);
    if (p.merge_tracks) {
      if (!p.global_tracking) for (int i = kKernelsPerEvent; i < kKernelsPerEvent + kKernelsGlobal; ++i) mark(ev, i, st);
      launch_merge(p, st, ev);
    }
    if (le == cudaSuccess) le = cudaGetLastError();
    if (capture) {
      cudaGraph_t g = nullptr;
      const cudaError_t ce = cudaStreamEndCapture(st, &g);      // always ends the capture, also after a failed launch
      if (le == cudaSuccess) le = ce;
      if (le == cudaSuccess) le = cudaGraphInstantiate(&gk->graph, g, 0);
      if (g) (void)cudaGraphDestroy(g);
      if (le != cudaSuccess) { gk->graph = nullptr; gk->seen = 0; return cuda_fail(le, "capture of the launch set"); }
      ++sl.n_captures;
      CU(cudaGraphLaunch(gk->graph, st));
    } else if (le != cudaSuccess) {
      return cuda_fail(le, "launch set");
    }
  }
  CU(cudaEventRecord(sl.ev_done, st));
  CU(cudaMemcpyAsync(sl.h_ctr, p.ctr, sizeof(Counters), cudaMemcpyDeviceToHost, st));
  CU(cudaEventRecord(sl.ev_ctr, st));   // counters are on the host
  sl.busy = true;
  return TPCST_OK;
}

int tpcst_wait_event(tpcst_ctx* ctx, int s, tpcst_tracks* out) {
  if (!ctx || !out || s < 0 || s >= TPCST_N_SLOTS) return TPCST_ERR_ARG;
  Slot& sl = ctx->slot[s];
  if (!sl.busy) return TPCST_ERR_STATE;
  GUARD(ctx);
  sl.busy = false;
  std::memset(out, 0, sizeof(*out));
  CU(cudaEventSynchronize(sl.ev_ctr));
  const Counters c = *sl.h_ctr;
  sl.done = true;
  sl.failed = c.error != 0u;
  if (c.error & kErrArg) return TPCST_ERR_ARG;       // device row_start: row_start[0] != 0 or row_start[last] != n_clusters
  if (c.error & kErrRange) return TPCST_ERR_RANGE;
  if (c.error & (kErrTrackletCap | kErrTrackCap)) return TPCST_ERR_CAPACITY;
  const Params& p = sl.m.prm;
  if (c.n_tracks) CU(cudaMemcpyAsync(sl.h_tracks, p.out_tracks, (size_t)c.n_tracks * sizeof(tpcst_track), cudaMemcpyDeviceToHost, ctx->st_d2h));
  if (c.n_ids) CU(cudaMemcpyAsync(sl.h_ids, p.out_ids, (size_t)c.n_ids * 4, cudaMemcpyDeviceToHost, ctx->st_d2h));
  if (p.global_tracking && c.n_global) {
    CU(cudaMemcpyAsync(sl.h_global, p.out_global, (size_t)c.n_global * sizeof(tpcst_global_ext), cudaMemcpyDeviceToHost, ctx->st_d2h));
    CU(cudaMemcpyAsync(sl.h_global_ids, p.out_global_ids, (size_t)c.n_global_ids * 4, cudaMemcpyDeviceToHost, ctx->st_d2h));
  }
  if (p.merge_tracks && c.n_tracks)
    CU(cudaMemcpyAsync(sl.h_merge, p.mg_seg, (size_t)c.n_tracks * sizeof(tpcst_merge_seg), cudaMemcpyDeviceToHost, ctx->st_d2h));
  CU(cudaStreamSynchronize(ctx->st_d2h));
  float ms = 0.f;
  CU(cudaEventElapsedTime(&ms, sl.ev_start, sl.ev_done));
  out->n_tracks = c.n_tracks; out->tracks = sl.h_tracks;
  out->n_cluster_ids = c.n_ids; out->cluster_ids = sl.h_ids;
  out->n_tracklets = c.n_tracklets; out->gpu_ms = ms;
  out->n_global = c.n_global; out->global_ext = sl.h_global;
  out->n_global_cluster_ids = c.n_global_ids; out->global_cluster_ids = sl.h_global_ids;
  out->n_merge = p.merge_tracks ? c.n_tracks : 0u; out->merge = sl.h_merge;
  return TPCST_OK;
}

int tpcst_track_event(tpcst_ctx* ctx, const tpcst_clusters* cl, tpcst_tracks* out) {
  const int rc = tpcst_submit_event(ctx, cl, 0);
  if (rc != TPCST_OK) return rc;
  return tpcst_wait_event(ctx, 0, out);
}

int tpcst_kernels_per_event(const tpcst_ctx* ctx) {
  if (ctx && ctx->cuts.merge_tracks) return kKernelsMax;
  return ctx && ctx->cuts.global_tracking ? kKernelsPerEvent + kKernelsGlobal : kKernelsPerEvent;
}
const char* tpcst_kernel_name(int i) { return kernel_name(i); }
int tpcst_set_profiling(tpcst_ctx* ctx, int on) {
  if (!ctx) return TPCST_ERR_ARG;
  if (on < 0 || on > 2) return TPCST_ERR_ARG;
  ctx->profiling = on;
  return TPCST_OK;
}

int tpcst_set_graphs(tpcst_ctx* ctx, int on) {
  if (!ctx || on < 0 || on > 1) return TPCST_ERR_ARG;
  ctx->graphs = on;
  return TPCST_OK;
}

int tpcst_selftest_math(void* stream, uint64_t n_div_pairs, uint64_t* n_checked, uint64_t* n_bad) {
  if (!n_checked || !n_bad) return TPCST_ERR_ARG;
  cudaStream_t st = (cudaStream_t)stream;
  unsigned long long* d_bad = nullptr;
  unsigned long long h_bad = 0;
  CU(cudaMalloc((void**)&d_bad, sizeof(*d_bad)));
  cudaError_t e = cudaMemsetAsync(d_bad, 0, sizeof(*d_bad), st);
  if (e == cudaSuccess) e = launch_selftest_math(n_div_pairs, d_bad, st);
  if (e == cudaSuccess) e = cudaMemcpyAsync(&h_bad, d_bad, sizeof(h_bad), cudaMemcpyDeviceToHost, st);
  if (e == cudaSuccess) e = cudaStreamSynchronize(st);
  (void)cudaFree(d_bad);
  if (e != cudaSuccess) return cuda_fail(e, "tpcst_selftest_math");
  *n_checked = (uint64_t)(0x43800000u - 0x3b800000u) + n_div_pairs;
  *n_bad = h_bad;
  return TPCST_OK;
}

const char* tpcst_error_string(int status) {
  switch (status) {
    case TPCST_OK: return "ok";
    case TPCST_ERR_ARG: return "bad argument";
    case TPCST_ERR_RANGE: return "a row holds more than 65535 clusters or its grid has too many bins";
    case TPCST_ERR_CAPACITY: return "workspace capacity exceeded (clusters, tracklets or tracks)";
    case TPCST_ERR_CUDA: return g_cuda_err;
    case TPCST_ERR_STATE: return "slot state: nothing submitted, or still busy";
    case TPCST_ERR_STATIC_LIMIT:
      return "tpcst_select_owners_static: more than TPCST_STATIC_MAX_CLUSTERS (1048576) clusters do not fit the library's "
             "fixed scratch array; select through tpcst_create / tpcst_track_event with a caller-allocated workspace instead";
  }
  return "unknown status";
}

int tpcst_destroy(tpcst_ctx* ctx) {
  if (!ctx) return TPCST_ERR_ARG;
  DeviceGuard guard(ctx->device);
  (void)cudaStreamSynchronize(ctx->st_compute);
  (void)cudaStreamSynchronize(ctx->st_copy);
  for (int i = 0; i < TPCST_N_SLOTS; ++i) {
    if (ctx->st_slot[i]) { (void)cudaStreamSynchronize(ctx->st_slot[i]); (void)cudaStreamDestroy(ctx->st_slot[i]); }
    if (ctx->ev_dep[i]) (void)cudaEventDestroy(ctx->ev_dep[i]);
  }
  if (ctx->st_d2h) { (void)cudaStreamSynchronize(ctx->st_d2h); (void)cudaStreamDestroy(ctx->st_d2h); }
  for (Slot& sl : ctx->slot) {
    if (sl.h_tracks) (void)cudaFreeHost(sl.h_tracks);
    if (sl.h_ids) (void)cudaFreeHost(sl.h_ids);
    if (sl.h_global) (void)cudaFreeHost(sl.h_global);
    if (sl.h_global_ids) (void)cudaFreeHost(sl.h_global_ids);
    if (sl.h_merge) (void)cudaFreeHost(sl.h_merge);
    if (sl.h_ctr) (void)cudaFreeHost(sl.h_ctr);
    for (Slot::GraphKey& k : sl.gkey) if (k.graph) (void)cudaGraphExecDestroy(k.graph);
    if (sl.ev_h2d) (void)cudaEventDestroy(sl.ev_h2d);
    if (sl.ev_ctr) (void)cudaEventDestroy(sl.ev_ctr);
    if (sl.ev_start) (void)cudaEventDestroy(sl.ev_start);
    if (sl.ev_done) (void)cudaEventDestroy(sl.ev_done);
    for (cudaEvent_t ek : sl.ev_k) if (ek) (void)cudaEventDestroy(ek);
  }
  delete ctx;
  return TPCST_OK;
}

// ---------------------------------------------------------------------------------------------
// Debug accessors: copy intermediate arrays to the host and convert sorted positions to the
// caller's cluster indices.  Slow by design (synchronous copies); used only by the parity tests.
int tpcst_debug_fetch(tpcst_ctx* ctx, int s, int what, void* host_buf, size_t cap, size_t* written) {
  if (!ctx || !written || s < 0 || s >= TPCST_N_SLOTS) return TPCST_ERR_ARG;
  Slot& sl = ctx->slot[s];
  if (!sl.done || sl.busy) return TPCST_ERR_STATE;
  GUARD(ctx);
  const Plan& pl = ctx->plan;
  const Params& p = sl.m.prm;
  const uint32_t N = sl.n_clusters, R = pl.R, SR = pl.SR;
  // the two measurement accessors touch nothing on the device: the slot's events have completed
  // and its counters are already on the host, so they are safe while the other slot is in flight
  if (what == TPCST_DBG_KERNEL_MS) {
    const int nk = tpcst_kernels_per_event(ctx);
    *written = sizeof(float) * nk;
    if (!sl.profiled) return TPCST_ERR_STATE;
    if (!host_buf || cap < *written) return TPCST_ERR_ARG;
    float* o = (float*)host_buf;
    for (int i = 0; i < nk; ++i) CU(cudaEventElapsedTime(&o[i], sl.ev_k[i], sl.ev_k[i + 1]));
    return TPCST_OK;
  }
  if (what == TPCST_DBG_WORK) {
    *written = 8 * sizeof(uint64_t);
    if (!sl.counted) return TPCST_ERR_STATE;
    if (!host_buf || cap < *written) return TPCST_ERR_ARG;
    const Counters& hc = *sl.h_ctr;
    const uint64_t v[8] = {hc.nf_window_tests, hc.nf_pair_evals, hc.kf_row_steps, hc.kf_searches,
                           hc.kf_candidates, hc.kf_updates, hc.claimed_hits, 0};
    std::memcpy(host_buf, v, sizeof(v));
    return TPCST_OK;
  }
  CU(cudaDeviceSynchronize());
  Counters c;
  CU(cudaMemcpy(&c, p.ctr, sizeof(c), cudaMemcpyDeviceToHost));
  // After a failed event only the counters (with the error bits) can be read: the kernels left early, so the intermediate
  // arrays are stale or half written, and the row_start of a TPCST_DEVICE event that failed its validation would be used
  // below to index host vectors and the caller's buffer.
  if (sl.failed && what != TPCST_DBG_COUNTERS) { *written = 0; return TPCST_ERR_STATE; }
  const uint32_t T = c.n_tracklets;
  std::vector<uint32_t> rs(SR + 1);
  CU(cudaMemcpy(rs.data(), p.row_start, (size_t)(SR + 1) * 4, cudaMemcpyDeviceToHost));
  auto need = [&](size_t bytes) -> bool { *written = bytes; return host_buf && cap >= bytes; };
  auto fetch_orig = [&](std::vector<uint32_t>& orig) -> int {
    orig.resize(pl.npad);
    CU(cudaMemcpy(orig.data(), p.s_orig, (size_t)pl.npad * 4, cudaMemcpyDeviceToHost));
    return TPCST_OK;
  };
  switch (what) {
    case TPCST_DBG_COUNTERS: {
      if (!need(32)) return TPCST_ERR_ARG;
      uint32_t v[8] = {N, c.n_tracklets, c.n_tracks, c.n_ids, c.error, sl.n_captures, sl.n_replays, 0};
      std::memcpy(host_buf, v, 32);
      return TPCST_OK;
    }
    case TPCST_DBG_BIN_OF: {
      if (!need((size_t)N * 4)) return TPCST_ERR_ARG;
      uint32_t* o = (uint32_t*)host_buf;
      CU(cudaMemcpy(o, p.bin_of, (size_t)N * 4, cudaMemcpyDeviceToHost));
      for (uint32_t i = 0; i < N; ++i) o[i] &= 0xffffu;
      return TPCST_OK;
    }
    case TPCST_DBG_BIN_START: {
      size_t tot = 0;
      for (uint32_t k = 0; k < R; ++k) tot += (size_t)pl.tab[k].ny * pl.nz;
      tot *= pl.S;
      if (!need(tot * 4)) return TPCST_ERR_ARG;
      std::vector<uint16_t> b((size_t)pl.S * pl.bins_sector_stride);
      CU(cudaMemcpy(b.data(), p.bins, b.size() * 2, cudaMemcpyDeviceToHost));
      uint32_t* o = (uint32_t*)host_buf;
      size_t w = 0;
      for (uint32_t sec = 0; sec < pl.S; ++sec)
        for (uint32_t k = 0; k < R; ++k) {
          const uint16_t* t = b.data() + (size_t)sec * pl.bins_sector_stride + pl.tab[k].bin_off;
          const uint32_t nb = pl.tab[k].ny * pl.nz;
          for (uint32_t i = 0; i < nb; ++i) o[w++] = t[i];
        }
      return TPCST_OK;
    }
    case TPCST_DBG_LINKS_RAW:
    case TPCST_DBG_LINKS: {
      if (!need((size_t)N * 8)) return TPCST_ERR_ARG;
      std::vector<uint32_t> orig;
      int rc = fetch_orig(orig);
      if (rc) return rc;
      std::vector<int32_t> up(pl.npad), dn(pl.npad);
      CU(cudaMemcpy(up.data(), what == TPCST_DBG_LINKS ? p.up : p.up_raw, (size_t)pl.npad * 4, cudaMemcpyDeviceToHost));
      CU(cudaMemcpy(dn.data(), what == TPCST_DBG_LINKS ? p.dn : p.dn_raw, (size_t)pl.npad * 4, cudaMemcpyDeviceToHost));
      int32_t* o = (int32_t*)host_buf;
      for (uint32_t sr = 0; sr < SR; ++sr) {
        const uint32_t p0 = pstart(rs[sr], sr), n = rs[sr + 1] - rs[sr];
        for (uint32_t i = 0; i < n; ++i) {
          const uint32_t g = orig[p0 + i];
          o[g] = up[p0 + i] >= 0 ? (int32_t)orig[up[p0 + i]] : -1;
          o[N + g] = dn[p0 + i] >= 0 ? (int32_t)orig[dn[p0 + i]] : -1;
        }
      }
      return TPCST_OK;
    }
    case TPCST_DBG_STARTS: {
      if (!need((size_t)T * 8)) return TPCST_ERR_ARG;
      std::vector<uint32_t> orig;
      int rc = fetch_orig(orig);
      if (rc) return rc;
      std::vector<uint32_t> sl_(pl.npad), ro(SR + 1);
      std::vector<int32_t> up(pl.npad);
      CU(cudaMemcpy(sl_.data(), p.start_list, (size_t)pl.npad * 4, cudaMemcpyDeviceToHost));
      CU(cudaMemcpy(up.data(), p.up, (size_t)pl.npad * 4, cudaMemcpyDeviceToHost));
      CU(cudaMemcpy(ro.data(), p.row_off, (size_t)(SR + 1) * 4, cudaMemcpyDeviceToHost));
      uint32_t* o = (uint32_t*)host_buf;
      for (uint32_t sr = 0; sr < SR; ++sr) {
        const uint32_t p0 = pstart(rs[sr], sr);
        for (uint32_t j = 0; j < ro[sr + 1] - ro[sr]; ++j) {
          o[ro[sr] + j] = orig[sl_[p0 + j]];
          uint32_t len = 1;                          // chain length: the device only checks >= min_chain
          for (int32_t c = up[sl_[p0 + j]]; c >= 0 && len < 65535u; c = up[c]) ++len;
          o[T + ro[sr] + j] = len;
        }
      }
      return TPCST_OK;
    }
    case TPCST_DBG_TRACKLETS: {
      if (!need((size_t)T * sizeof(tpcst_track))) return TPCST_ERR_ARG;
      std::vector<uint32_t> orig;
      int rc = fetch_orig(orig);
      if (rc) return rc;
      std::vector<uint32_t> rows(T), seed(T), kept(T), ro(SR + 1), ref;
      if (p.t_ref) { ref.resize(T); CU(cudaMemcpy(ref.data(), p.t_ref, (size_t)T * 4, cudaMemcpyDeviceToHost)); }
      std::vector<float> chi2(T), par((size_t)5 * pl.tcap), cov((size_t)9 * pl.tcap);
      CU(cudaMemcpy(rows.data(), p.t_rows, (size_t)T * 4, cudaMemcpyDeviceToHost));
      CU(cudaMemcpy(seed.data(), p.t_seed, (size_t)T * 4, cudaMemcpyDeviceToHost));
      CU(cudaMemcpy(kept.data(), p.t_kept, (size_t)T * 4, cudaMemcpyDeviceToHost));
      CU(cudaMemcpy(chi2.data(), p.t_chi2, (size_t)T * 4, cudaMemcpyDeviceToHost));
      CU(cudaMemcpy(par.data(), p.t_par, par.size() * 4, cudaMemcpyDeviceToHost));
      CU(cudaMemcpy(cov.data(), p.t_cov, cov.size() * 4, cudaMemcpyDeviceToHost));
      CU(cudaMemcpy(ro.data(), p.row_off, (size_t)(SR + 1) * 4, cudaMemcpyDeviceToHost));
      tpcst_track* o = (tpcst_track*)host_buf;
      const size_t hs = pl.tcap;
      uint32_t sr = 0;
      for (uint32_t t = 0; t < T; ++t) {
        while (ro[sr + 1] <= t) ++sr;
        tpcst_track& k = o[t];
        std::memset(&k, 0, sizeof(k));
        k.sector = sr / R; k.first_row = rows[t] & 0xffu; k.last_row = (rows[t] >> 8) & 0xffu;
        k.n_clusters = (rows[t] >> 16) & 0xffu; k.first_cluster = kept[t] & 0x7fffffffu; k.seed_cluster = orig[seed[t]];
        k.x_ref = pl.tab[ref.empty() ? k.first_row : ref[t]].x;
        k.y = par[t]; k.z = par[hs + t]; k.sinphi = par[2 * hs + t]; k.dzds = par[3 * hs + t];
        k.qpt = (0.0f - par[4 * hs + t]) / ctx->kbz;
        k.cov[0] = cov[t]; k.cov[3] = cov[hs + t]; k.cov[5] = cov[2 * hs + t]; k.cov[10] = cov[3 * hs + t];
        k.cov[12] = cov[4 * hs + t]; k.cov[14] = cov[5 * hs + t]; k.cov[2] = cov[6 * hs + t];
        k.cov[7] = cov[7 * hs + t]; k.cov[9] = cov[8 * hs + t];
        k.chi2 = chi2[t];
      }
      return TPCST_OK;
    }
    case TPCST_DBG_ROW_HITS: {
      if (!need((size_t)T * R * 4)) return TPCST_ERR_ARG;
      std::vector<uint32_t> orig;
      int rc = fetch_orig(orig);
      if (rc) return rc;
      std::vector<uint32_t> rows(T);
      CU(cudaMemcpy(rows.data(), p.t_rows, (size_t)T * 4, cudaMemcpyDeviceToHost));
      std::vector<uint16_t> h((size_t)T * pl.hit_stride);
      if (T) CU(cudaMemcpy(h.data(), p.hits, h.size() * 2, cudaMemcpyDeviceToHost));
      int32_t* o = (int32_t*)host_buf;
      for (size_t i = 0; i < (size_t)T * R; ++i) o[i] = -1;
      std::vector<uint32_t> ro(SR + 1);
      CU(cudaMemcpy(ro.data(), p.row_off, (size_t)(SR + 1) * 4, cudaMemcpyDeviceToHost));
      uint32_t sr = 0;
      for (uint32_t t = 0; t < T; ++t) {
        while (ro[sr + 1] <= t) ++sr;
        const uint32_t sec = sr / R, first = rows[t] & 0xffu, last = (rows[t] >> 8) & 0xffu;
        for (uint32_t k = first; k <= last && k < R; ++k) {
          const uint16_t v = h[(size_t)t * pl.hit_stride + k];
          if (v != 0xffffu) o[(size_t)t * R + k] = (int32_t)orig[pstart(rs[sec * R + k], sec * R + k) + v];
        }
      }
      return TPCST_OK;
    }
    case TPCST_DBG_OWNERS: {
      if (!need((size_t)N * 4)) return TPCST_ERR_ARG;
      launch_owners_to_orig(p, ctx->d_dbg, ctx->st_compute);
      CU(cudaStreamSynchronize(ctx->st_compute));
      CU(cudaMemcpy(host_buf, ctx->d_dbg, (size_t)N * 4, cudaMemcpyDeviceToHost));
      return TPCST_OK;
    }
  }
  return TPCST_ERR_ARG;
}

}  // extern "C"
