// oracle/tpc_oracle.cpp — CPU oracle of the ALICE HLT TPC sector tracker (arXiv 1712.09407).
//
// TEST INFRASTRUCTURE ONLY.  This file is the slow, plain, single-purpose CPU statement of what
// the hot path computes.  Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline /
// --impl reference legs may build, load or call it.  It shares no code, header, table generator
// or helper with paper_1712_09407_b200/ (the CUDA path); neither includes the other.
//
// What it follows.  PAPER.md §1 L36-L46 gives the method in words: neighbours finder (L40),
// evolution step (L41), tracklets = chains of one-to-one links (L43), Kalman tracklet construction
// (L45), tracklet selection (L46, first-wins rule L78, minimum 30 clusters L116), output = a list
// of clusters per track (L102).  The paper prints no formula, constant (except 30 and alpha = 6),
// pseudo-code or worked example for these steps, so every quantitative choice is a *reading*,
// listed as G1..G32 in DESIGN.md §"Readings of the paper"; the comments below cite both.
//
// Pins (tests/test_oracle_*.py): geometry closed forms; binning invariants; neighbours finder ==
// brute-force enumeration of all (u, d) triplets (MODE_TRIPLET, the plain definition) and
// independent of the grid; links follow truth on noise-free straight/helix tracks; evolution
// reciprocity; chain invariants; transport == analytic helix; update == textbook Kalman update;
// the whole construction with kappa frozen == the weighted least-squares straight-line fit of the
// same clusters (closed form, both passes, covariance and chi2); the stop rules, the miss counters
// and the truncation rule of construct_sector on hand-worked single-track events with gaps
// (test_oracle_construction_rules.py); noise-free helix parameters recovered; chi2/pull statistics;
// selection == sequential greedy reference (length rule) and == sequential weight-ordered
// reference (mode 1); no shared clusters; length >= cut; the G29 near-threshold log (bisection on the
// displacement at which a pickup flips; grid == row scan); global tracking: rotation == exact
// geometry, hand-worked prolongations (gap rule, free clusters only, edge and row limits).
// Parity unpinned (free parameters with no value in the paper): the cut defaults themselves.
//
// Arithmetic: all tracker arithmetic is IEEE binary32, one rounding per written operation, in the
// association written here (build with -O2 -ffp-contract=off, never -ffast-math).  Derived tables
// are (float)(double expression) so that an independent implementation can agree bit for bit.

#include <algorithm>
#include <atomic>
#include <cmath>
#include <cstdint>
#include <cstring>
#include <thread>
#include <vector>

namespace {

struct Geometry {            // mirrors the ctypes struct in oracle/oracle.py
  uint32_t n_sectors, n_rows;
  const float* row_x;
  float tan_half_angle, z_max, bz_tesla;
};

struct Cuts {                // every free parameter of the readings, fp32
  float bin_y, bin_z, grid_pad;                                    // G4
  float nf_wy_slope, nf_wy_const, nf_wz_slope, nf_wz_const;        // G6
  float nf_max_dev2;                                               // G7
  uint32_t min_chain_clusters;                                     // G12
  float err_y2, err_z2;                                            // G17
  float q_sinphi, q_dzds;                                          // G18
  float c0_sinphi, c0_dzds, c0_kappa;                              // G15
  float max_sinphi;                                                // G16b
  float chi2_cut;                                                  // G20
  uint32_t max_row_gap;                                            // G21
  float edge_margin;                                               // G23
  uint32_t min_clusters;                                           // L116 / G26
  float min_pt;                                                    // L46 / G26
  uint32_t select_mode;      // 0 = longest wins (L46, L78); 1 = chi2-weighted (L80-L94, NEXT-1)
  float alpha;               // L94: 6
  uint32_t global_tracking;  // NEXT-2 (L116-L136): 1 = prolong track ends into the neighbouring sector (G33-G36)
  uint32_t gt_max_rows;      // G33: an end qualifies if at most this many rows lie beyond it (default 30 = L116)
  float gt_edge;             // G33: ... and it lies within this distance of the sector edge [cm]
  uint32_t select_rounds;    // G26b (NEXT-4, L46): 2 = clusters of tracklets that fail the cuts are released and claimed again
  uint32_t merge_tracks;     // NEXT-3 (L28, L98, L102): 1 = sort, refit and link the sector tracks (G37-G40)
  uint32_t merge_max_gap;    // G39: rows between the end of a segment and the start of its continuation, at most
  float merge_chi2_cut;      // G39: cut on the 5-parameter match chi2
  uint32_t max_passes;       // G22d (NEXT-4, L45 "repeated until no more clusters are found"): passes over the tracklet, >= 2
};

enum { MODE_GRID = 0, MODE_ROWSCAN = 1, MODE_TRIPLET = 2 };   // neighbours finder / pickup search

struct Track {               // mirrors oracle.py TRACK_DTYPE (not the CUDA library's struct)
  uint32_t sector, first_row, last_row, n_clusters, first_cluster, seed_cluster;
  float x_ref, y, z, sinphi, dzds, qpt;
  float cov[15];
  float chi2;
};

struct GlobalExt {           // NEXT-2 output record (G36); mirrors oracle.py GLOBAL_DTYPE
  uint32_t track, sector, end, n_clusters, first_cluster, row;   // end: 0 = inner (prolonged downwards), 1 = outer
  float x_ref, y, z, sinphi, dzds, qpt;
  float cov[15];
  float chi2;
};

struct Tables {              // derived per-row tables, (float)(double expr) — DESIGN.md "Derived tables"
  std::vector<float> x, ymax, ratio_up, ratio_dn, w_up, w_dn, wy_up, wy_dn, wz_up, wz_dn;
  std::vector<uint32_t> ny;
  uint32_t nz;
  float inv_bin_y, inv_bin_z, kbz, max_qpt;
  float gt_cos, gt_sin;      // cos / sin of the angle between neighbouring sectors, 2 atan(tan_half_angle)
};

struct Counters {            // work counters for the roofline arithmetic
  uint64_t nf_window_tests = 0, nf_pair_evals = 0, links_raw = 0, links_evolved = 0, starts = 0;
  uint64_t kf_row_steps = 0, kf_candidates = 0, kf_updates = 0, claimed_hits = 0, tracks = 0, track_clusters = 0;
};

struct SectorResult {
  // per cluster arrays are written straight into the event-level arrays (disjoint ranges)
  std::vector<uint32_t> start_cluster, chain_len;
  std::vector<uint32_t> first_row, last_row, nhits;
  std::vector<uint32_t> ref_row, n_passes;       // row the parameters are given at; passes that shaped the tracklet (G22d)
  std::vector<float> params, cov, chi2;          // [T*5], [T*15], [T]
  std::vector<float> top;                        // [T*20] state + covariance at the top hit row, end of the up pass (G36)
  std::vector<int32_t> hits;                     // [T*R] global original index or -1
  std::vector<uint32_t> kept;                    // [T] clusters owned after selection
  std::vector<uint8_t> accepted;                 // [T]
  std::vector<uint32_t> near;                    // G29 audit: (tracklet of the sector, row) of every near-threshold pickup decision
  Counters cnt;
};

struct MergeSeg {            // NEXT-3 output record, one per track (G37-G40); mirrors oracle.py MERGE_DTYPE
  uint32_t rank;             // position of the track in the merger's canonical order (G37)
  int32_t next, prev;        // track that continues this one in the neighbouring sector / that it continues; -1 = none
  uint32_t ok;               // 1 = both refit passes completed (G38)
  uint32_t row_in, row_out;  // rows of the first and of the last cluster of the list: where the two states are given
  float chi2, match_chi2;    // inward-pass chi2; chi2 of the kept link to `next`
  float in_par[5], in_cov[15], out_par[5], out_cov[15];   // (y, z, sin phi, dz/ds, kappa) at row_x[row_in] / row_x[row_out]
  // G41, at the first segment of every chain (prev == -1), else zero: the merged track
  uint32_t chain_n_seg, chain_n_clusters;                 // segments and clusters of the chain; n_seg = 0: not a head, or the joint refit failed
  float chain_chi2;                                       // inward-pass chi2 of the joint refit
  float chain_par[5], chain_cov[15];                      // state at row_x[row_in] of the head, in the head's frame
};
struct MergeCand { uint32_t a, b; float chi2; };          // every accepted (segment, continuation) pair (tests)

struct Oracle {
  Geometry geo;
  std::vector<float> row_x;
  Cuts cuts;
  Tables tab;
  // event-level results (original-index space)
  uint32_t n = 0;
  std::vector<uint32_t> row_start;
  std::vector<uint32_t> bin_of, bin_row_offset, bin_count, bin_start;
  std::vector<int32_t> up_raw, dn_raw, up, dn;
  std::vector<uint32_t> owner;
  std::vector<uint32_t> start_cluster, chain_len, first_row, last_row, nhits, kept, tracklet_sector, ref_row, n_passes;
  std::vector<uint32_t> near;                    // G29 audit: (tracklet id, row) pairs
  std::vector<uint8_t> accepted;
  std::vector<float> params, cov, chi2;
  std::vector<int32_t> hits;
  std::vector<Track> tracks;
  std::vector<uint32_t> track_cluster_ids;
  std::vector<GlobalExt> global_ext;             // NEXT-2
  std::vector<uint32_t> global_cluster_ids;
  std::vector<MergeSeg> merge;                   // NEXT-3
  std::vector<MergeCand> merge_cand;
  Counters cnt;
};

// ---------------------------------------------------------------------------------------------
// Derived tables (G1, G4, G6, G7).  Each entry is a double expression of the fp32 inputs, rounded
// once to fp32.
void build_tables(Oracle& o) {
  const uint32_t R = o.geo.n_rows;
  Tables& t = o.tab;
  const Cuts& c = o.cuts;
  t.x = o.row_x;
  t.ymax.assign(R, 0.f); t.ratio_up.assign(R, 0.f); t.ratio_dn.assign(R, 0.f);
  t.w_up.assign(R, 0.f); t.w_dn.assign(R, 0.f);
  t.wy_up.assign(R, 0.f); t.wy_dn.assign(R, 0.f); t.wz_up.assign(R, 0.f); t.wz_dn.assign(R, 0.f);
  t.ny.assign(R, 1);
  for (uint32_t k = 0; k < R; ++k) {
    const double xk = (double)t.x[k];
    t.ymax[k] = (float)(xk * (double)o.geo.tan_half_angle);
    t.ny[k] = (uint32_t)std::ceil(2.0 * (double)t.ymax[k] / (double)c.bin_y) + 1u;              // G4
    if (k + 1 < R) {
      const double xu = (double)t.x[k + 1];
      t.ratio_up[k] = (float)(xu / xk);
      t.wy_up[k] = (float)((double)c.nf_wy_slope * (xu - xk) + (double)c.nf_wy_const);           // G6
      t.wz_up[k] = (float)((double)c.nf_wz_slope * (xu - xk) + (double)c.nf_wz_const);
    }
    if (k > 0) {
      const double xd = (double)t.x[k - 1];
      t.ratio_dn[k] = (float)(xd / xk);
      t.wy_dn[k] = (float)((double)c.nf_wy_slope * (xk - xd) + (double)c.nf_wy_const);
      t.wz_dn[k] = (float)((double)c.nf_wz_slope * (xk - xd) + (double)c.nf_wz_const);
    }
    if (k > 0 && k + 1 < R) {                                                                     // G7
      const double xu = (double)t.x[k + 1], xd = (double)t.x[k - 1];
      t.w_up[k] = (float)((xk - xd) / (xu - xd));
      t.w_dn[k] = (float)((xu - xk) / (xu - xd));
    }
  }
  t.nz = (uint32_t)std::ceil((double)o.geo.z_max / (double)c.bin_z) + 1u;
  t.inv_bin_y = (float)(1.0 / (double)c.bin_y);
  t.inv_bin_z = (float)(1.0 / (double)c.bin_z);
  t.kbz = (float)(0.299792458e-2 * (double)o.geo.bz_tesla);                                       // G14
  t.max_qpt = (float)(1.0 / (double)c.min_pt);
  const double dphi = 2.0 * std::atan((double)o.geo.tan_half_angle);   // G34: angle between neighbouring sectors
  t.gt_cos = (float)std::cos(dphi); t.gt_sin = (float)std::sin(dphi);
}

// G4: bin coordinate.  f = (v + off) * inv; clamp to [0, n-1]; truncation toward zero.  NaN -> 0.
inline uint32_t bin_coord(float v, float off, float inv, uint32_t n) {
  const float f = (v + off) * inv;
  if (!(f >= 0.0f)) return 0u;
  if (f >= (float)(n - 1u)) return n - 1u;
  return (uint32_t)f;
}

// A row's view: clusters [g0, g1) in original order plus its grid.
struct RowView {
  uint32_t g0, g1, ny, nz;
  float ymax;
  const uint32_t* bstart;        // [ny*nz] exclusive start within row
  const uint32_t* bcount;
  const uint32_t* sorted;        // [n] global original indices in (bin, original index) order
};

struct SectorCtx {
  const Oracle* o;
  const float* xyz;
  uint32_t sector;
  std::vector<RowView> rows;
  std::vector<uint32_t> sorted;  // concatenated per row, indexed (g - sector_g0)
  uint32_t g_base;
  int mode;
  inline float Y(uint32_t g) const { return xyz[3 * (size_t)g + 1]; }
  inline float Z(uint32_t g) const { return xyz[3 * (size_t)g + 2]; }
};

// ---------------------------------------------------------------------------------------------
// Step 1 — grid binning (paper: "initialization", L52; north_star step 1; reading G4/G5).
void bin_sector(Oracle& o, SectorCtx& sc) {
  const uint32_t R = o.geo.n_rows;
  const Tables& t = o.tab;
  sc.rows.resize(R);
  sc.g_base = o.row_start[sc.sector * R];
  sc.sorted.resize(o.row_start[(sc.sector + 1) * R] - sc.g_base);
  for (uint32_t k = 0; k < R; ++k) {
    const uint32_t sr = sc.sector * R + k;
    const uint32_t g0 = o.row_start[sr], g1 = o.row_start[sr + 1];
    const uint32_t ny = t.ny[k], nz = t.nz, nb = ny * nz;
    uint32_t* cnt = &o.bin_count[o.bin_row_offset[sr]];
    uint32_t* bst = &o.bin_start[o.bin_row_offset[sr]];
    std::fill(cnt, cnt + nb, 0u);
    for (uint32_t g = g0; g < g1; ++g) {
      const uint32_t iy = bin_coord(sc.Y(g), t.ymax[k], t.inv_bin_y, ny);
      const uint32_t iz = bin_coord(sc.Z(g), 0.0f, t.inv_bin_z, nz);
      const uint32_t b = iz * ny + iy;                       // y fastest
      o.bin_of[g] = b;
      ++cnt[b];
    }
    uint32_t acc = 0;
    for (uint32_t b = 0; b < nb; ++b) { bst[b] = acc; acc += cnt[b]; }
    std::vector<uint32_t> cur(bst, bst + nb);
    uint32_t* srt = sc.sorted.data() + (g0 - sc.g_base);
    for (uint32_t g = g0; g < g1; ++g) srt[cur[o.bin_of[g]]++] = g;   // stable: ascending original index per bin
    sc.rows[k] = RowView{g0, g1, ny, nz, t.ymax[k], bst, cnt, srt};
  }
}

// Visit every cluster of row `rv` whose bin intersects the box [ylo, yhi] x [zlo, zhi] widened by
// grid_pad (G4 "the grid is only an acceleration structure"), or the whole row in ROWSCAN mode.
template <class F>
inline void for_candidates(const SectorCtx& sc, const RowView& rv, float ylo, float yhi, float zlo, float zhi, F&& f) {
  if (sc.mode != MODE_GRID) {
    for (uint32_t g = rv.g0; g < rv.g1; ++g) f(g);
    return;
  }
  const Tables& t = sc.o->tab;
  const float pad = sc.o->cuts.grid_pad;
  const uint32_t iy0 = bin_coord(ylo - pad, rv.ymax, t.inv_bin_y, rv.ny);
  const uint32_t iy1 = bin_coord(yhi + pad, rv.ymax, t.inv_bin_y, rv.ny);
  const uint32_t iz0 = bin_coord(zlo - pad, 0.0f, t.inv_bin_z, rv.nz);
  const uint32_t iz1 = bin_coord(zhi + pad, 0.0f, t.inv_bin_z, rv.nz);
  for (uint32_t iz = iz0; iz <= iz1; ++iz) {
    const uint32_t b0 = iz * rv.ny + iy0, b1 = iz * rv.ny + iy1;
    const uint32_t p0 = rv.bstart[b0], p1 = rv.bstart[b1] + rv.bcount[b1];   // bins iy0..iy1 are contiguous
    for (uint32_t p = p0; p < p1; ++p) f(rv.sorted[p]);
  }
}

// ---------------------------------------------------------------------------------------------
// Step 2 — neighbours finder (L40, Fig. 3a; readings G6-G10, G32).
// For cluster c on row k: among up candidates u (row k+1) and down candidates d (row k-1) inside
// the search windows, the pair minimising the straight-line deviation D; ties -> smaller original
// index of u, then of d.  Both links or none.
inline bool in_window(float v, float centre, float w) { const float dv = v - centre; return std::fabs(dv) <= w; }

inline float deviation2(float y, float z, float yu, float zu, float yd, float zd, float wu, float wd) {
  const float t1 = yu * wu, t2 = yd * wd;
  const float ey = (t1 + t2) - y;
  const float s1 = zu * wu, s2 = zd * wd;
  const float ez = (s1 + s2) - z;
  return (ey * ey) + (ez * ez);                               // G7
}

void neighbours_sector(Oracle& o, SectorCtx& sc, Counters& cnt) {
  const uint32_t R = o.geo.n_rows;
  const Tables& t = o.tab;
  const float maxdev = o.cuts.nf_max_dev2;
  std::vector<uint32_t> U, Dn;
  for (uint32_t k = 0; k < R; ++k) {
    const RowView& rv = sc.rows[k];
    for (uint32_t g = rv.g0; g < rv.g1; ++g) { o.up_raw[g] = -1; o.dn_raw[g] = -1; }
    if (k == 0 || k + 1 >= R) continue;                       // G9: rows 0 and R-1 get no links
    const RowView& ru = sc.rows[k + 1];
    const RowView& rd = sc.rows[k - 1];
    const float wu = t.w_up[k], wd = t.w_dn[k];
    for (uint32_t g = rv.g0; g < rv.g1; ++g) {
      const float y = sc.Y(g), z = sc.Z(g);
      const float pyu = y * t.ratio_up[k], pzu = z * t.ratio_up[k];     // G6: projection from the origin
      const float pyd = y * t.ratio_dn[k], pzd = z * t.ratio_dn[k];
      float bestD = 0.f; int32_t bu = -1, bd = -1;
      auto consider = [&](uint32_t u, uint32_t d) {
        ++cnt.nf_pair_evals;
        const float D = deviation2(y, z, sc.Y(u), sc.Z(u), sc.Y(d), sc.Z(d), wu, wd);
        if (!(D <= maxdev)) return;
        if (bu < 0 || D < bestD || (D == bestD && ((int32_t)u < bu || ((int32_t)u == bu && (int32_t)d < bd)))) {
          bestD = D; bu = (int32_t)u; bd = (int32_t)d;       // G8
        }
      };
      if (sc.mode == MODE_TRIPLET) {                          // the plain definition: all (u, d) pairs
        for (uint32_t u = ru.g0; u < ru.g1; ++u)
          for (uint32_t d = rd.g0; d < rd.g1; ++d) {
            cnt.nf_window_tests += 2;
            if (!in_window(sc.Y(u), pyu, t.wy_up[k]) || !in_window(sc.Z(u), pzu, t.wz_up[k])) continue;
            if (!in_window(sc.Y(d), pyd, t.wy_dn[k]) || !in_window(sc.Z(d), pzd, t.wz_dn[k])) continue;
            consider(u, d);
          }
      } else {
        U.clear(); Dn.clear();
        for_candidates(sc, ru, pyu - t.wy_up[k], pyu + t.wy_up[k], pzu - t.wz_up[k], pzu + t.wz_up[k], [&](uint32_t u) {
          ++cnt.nf_window_tests;
          if (in_window(sc.Y(u), pyu, t.wy_up[k]) && in_window(sc.Z(u), pzu, t.wz_up[k])) U.push_back(u);
        });
        if (!U.empty())
          for_candidates(sc, rd, pyd - t.wy_dn[k], pyd + t.wy_dn[k], pzd - t.wz_dn[k], pzd + t.wz_dn[k], [&](uint32_t d) {
            ++cnt.nf_window_tests;
            if (in_window(sc.Y(d), pyd, t.wy_dn[k]) && in_window(sc.Z(d), pzd, t.wz_dn[k])) Dn.push_back(d);
          });
        for (uint32_t u : U) for (uint32_t d : Dn) consider(u, d);
      }
      o.up_raw[g] = bu; o.dn_raw[g] = bd;
      if (bu >= 0) cnt.links_raw += 2;
    }
  }
}

// ---------------------------------------------------------------------------------------------
// Step 3 — evolution (L41, Fig. 3b; G11): keep reciprocal links only, from a snapshot.
void evolve_sector(Oracle& o, const SectorCtx& sc, Counters& cnt) {
  const uint32_t R = o.geo.n_rows;
  const uint32_t g0 = o.row_start[sc.sector * R], g1 = o.row_start[(sc.sector + 1) * R];
  for (uint32_t g = g0; g < g1; ++g) {
    const int32_t u = o.up_raw[g], d = o.dn_raw[g];
    o.up[g] = (u >= 0 && o.dn_raw[u] == (int32_t)g) ? u : -1;
    o.dn[g] = (d >= 0 && o.up_raw[d] == (int32_t)g) ? d : -1;
    cnt.links_evolved += (o.up[g] >= 0) + (o.dn[g] >= 0);
  }
}

// ---------------------------------------------------------------------------------------------
// Step 5 helpers — Kalman state, transport (G16), update (G17, G19).
// State p = (y, z, s = sin phi, t = dz/ds, k = curvature) at the x of a row; covariance lower
// triangle c[i*(i+1)/2 + j], i >= j.
struct State { float y, z, s, t, k; float c[15]; };
inline float& C(State& st, int i, int j) { return i >= j ? st.c[i * (i + 1) / 2 + j] : st.c[j * (j + 1) / 2 + i]; }
inline float Cc(const State& st, int i, int j) { return i >= j ? st.c[i * (i + 1) / 2 + j] : st.c[j * (j + 1) / 2 + i]; }

// G16: exact circle transport in x-y by dx, series for the path length, Jacobian with dz'/ds and
// dz'/dk neglected.  nrows = number of row steps spanned (process noise G18 scales with it).
bool transport(const Cuts& cu, const State& a, float dx, float nrows, State& b) {
  const float s1 = a.s + a.k * dx;
  if (!(std::fabs(s1) <= cu.max_sinphi)) return false;       // G16b (also rejects NaN)
  const float cc = std::sqrt(1.0f - a.s * a.s);
  const float c1 = std::sqrt(1.0f - s1 * s1);
  const float ss = a.s + s1;
  const float cs = cc + c1;
  const float T = ss / cs;
  b.y = a.y + dx * T;
  const float L = dx * std::sqrt(1.0f + T * T);
  const float u = (a.k * L) * 0.5f;
  const float u2 = u * u;
  const float ser = 1.0f + (u2 * (1.0f / 6.0f) + (u2 * u2) * 0.075f);   // asin(u)/u
  const float ds = L * ser;
  b.z = a.z + a.t * ds;
  b.s = s1; b.t = a.t; b.k = a.k;
  const float r0 = a.s / cc, r1 = s1 / c1;
  const float d2 = cs * cs;
  const float h2 = (dx * ((2.0f * cs) + ss * (r0 + r1))) / d2;
  const float h4 = ((dx * dx) * (cs + ss * r1)) / d2;
  // M = F C with F = I + h2 E02 + h4 E04 + ds E13 + dx E24
  float M[5][5];
  for (int j = 0; j < 5; ++j) {
    M[0][j] = Cc(a, 0, j) + h2 * Cc(a, 2, j) + h4 * Cc(a, 4, j);
    M[1][j] = Cc(a, 1, j) + ds * Cc(a, 3, j);
    M[2][j] = Cc(a, 2, j) + dx * Cc(a, 4, j);
    M[3][j] = Cc(a, 3, j);
    M[4][j] = Cc(a, 4, j);
  }
  // C' = M F^T (lower triangle)
  for (int i = 0; i < 5; ++i) {
    C(b, i, 0) = M[i][0] + h2 * M[i][2] + h4 * M[i][4];
    if (i >= 1) C(b, i, 1) = M[i][1] + ds * M[i][3];
    if (i >= 2) C(b, i, 2) = M[i][2] + dx * M[i][4];
    if (i >= 3) C(b, i, 3) = M[i][3];
    if (i >= 4) C(b, i, 4) = M[i][4];
  }
  C(b, 2, 2) = Cc(b, 2, 2) + cu.q_sinphi * nrows;             // G18
  C(b, 3, 3) = Cc(b, 3, 3) + cu.q_dzds * nrows;
  return true;
}

struct InvS { float i00, i01, i11; };
// G17/G24: inverse of the 2x2 innovation covariance.
inline bool innovation(const Cuts& cu, const State& a, InvS& w, float& S00, float& S11) {
  S00 = Cc(a, 0, 0) + cu.err_y2;
  const float S01 = Cc(a, 1, 0);
  S11 = Cc(a, 1, 1) + cu.err_z2;
  const float det = S00 * S11 - S01 * S01;
  if (!(det > 0.0f) || !(S00 > 0.0f)) return false;
  w.i00 = S11 / det; w.i01 = (-S01) / det; w.i11 = S00 / det;
  return true;
}
inline float chi2_of(const InvS& w, float r0, float r1) {      // G19
  return ((r0 * r0) * w.i00 + (2.0f * (r0 * r1)) * w.i01) + (r1 * r1) * w.i11;
}
// G17: joint 2-D update with measurement (ym, zm); result in b.  Fails if |s| leaves the band.
bool update(const Cuts& cu, const State& a, const InvS& w, float ym, float zm, State& b) {
  const float r0 = ym - a.y, r1 = zm - a.z;
  float K0[5], K1[5];
  for (int i = 0; i < 5; ++i) {
    K0[i] = Cc(a, i, 0) * w.i00 + Cc(a, i, 1) * w.i01;
    K1[i] = Cc(a, i, 0) * w.i01 + Cc(a, i, 1) * w.i11;
  }
  b.y = a.y + (K0[0] * r0 + K1[0] * r1);
  b.z = a.z + (K0[1] * r0 + K1[1] * r1);
  b.s = a.s + (K0[2] * r0 + K1[2] * r1);
  b.t = a.t + (K0[3] * r0 + K1[3] * r1);
  b.k = a.k + (K0[4] * r0 + K1[4] * r1);
  if (!(std::fabs(b.s) <= cu.max_sinphi)) return false;
  for (int i = 0; i < 5; ++i)
    for (int j = 0; j <= i; ++j)
      C(b, i, j) = Cc(a, i, j) - (K0[i] * Cc(a, 0, j) + K1[i] * Cc(a, 1, j));
  return true;
}

inline void reset_cov(const Cuts& cu, State& st) {            // G15 diagonal prior
  for (float& v : st.c) v = 0.0f;
  C(st, 0, 0) = cu.err_y2; C(st, 1, 1) = cu.err_z2;
  C(st, 2, 2) = cu.c0_sinphi; C(st, 3, 3) = cu.c0_dzds; C(st, 4, 4) = cu.c0_kappa;
}

// G20 pickup: over the row (grid-accelerated or whole row) the cluster with minimal chi2, ties ->
// smaller original index.  Returns -1 if the row has no cluster; acceptance is the caller's.
// G29 audit: `near` is set when the decision on this row hangs on less than 1e-4 (relative): the smallest chi2 of
// the row lies within 1e-4 of the cut (above or below it), or the two smallest chi2 differ by less than 1e-4 of the
// smaller ("if within one row two clusters are equally close to the trajectory ... either the one or the other can
// get assigned", L102).  Bookkeeping only: it does not enter the result.
int32_t best_on_row(const SectorCtx& sc, const RowView& rv, const State& p, const InvS& w, float S00, float S11,
                    float& best_chi2, Counters& cnt, bool* near = nullptr) {
  const Cuts& cu = sc.o->cuts;
  const float by = std::sqrt(cu.chi2_cut * S00) * 1.001f;      // box contains the chi2 <= cut ellipse
  const float bz = std::sqrt(cu.chi2_cut * S11) * 1.001f;
  int32_t best = -1; best_chi2 = 0.f;
  double m1 = -1.0, m2 = -1.0;                                  // the two smallest chi2 among the visited clusters (audit)
  for_candidates(sc, rv, p.y - by, p.y + by, p.z - bz, p.z + bz, [&](uint32_t g) {
    ++cnt.kf_candidates;
    const float c2 = chi2_of(w, sc.Y(g) - p.y, sc.Z(g) - p.z);
    if (c2 == c2) {
      if (m1 < 0.0 || c2 < m1) { m2 = m1; m1 = c2; } else if (m2 < 0.0 || c2 < m2) m2 = c2;
    }
    if (!(c2 <= cu.chi2_cut)) return;                          // only clusters that pass can win
    if (best < 0 || c2 < best_chi2 || (c2 == best_chi2 && (int32_t)g < best)) { best = (int32_t)g; best_chi2 = c2; }
  });
  if (near) {
    const double cut = (double)cu.chi2_cut;
    *near = (m1 >= 0.0 && std::fabs(m1 - cut) <= 1e-4 * cut) || (m1 >= 0.0 && m2 >= 0.0 && m1 <= cut * (1.0 + 1e-4) && m2 - m1 <= 1e-4 * m1);
  }
  return best;
}

// ---------------------------------------------------------------------------------------------
// Steps 4-5 — tracklet starts/chains (L43; G12) and Kalman construction (L45; G14-G25).
void construct_sector(Oracle& o, const SectorCtx& sc, SectorResult& out) {
  const uint32_t R = o.geo.n_rows;
  const Cuts& cu = o.cuts;
  const Tables& t = o.tab;
  Counters& cnt = out.cnt;
  for (uint32_t k0 = 0; k0 < R; ++k0) {
    const RowView& rv = sc.rows[k0];
    for (uint32_t g = rv.g0; g < rv.g1; ++g) {
      if (!(o.up[g] >= 0 && o.dn[g] < 0)) continue;           // G12: start
      uint32_t len = 1;
      for (int32_t c = o.up[g]; c >= 0; c = o.up[c]) ++len;
      if (len < cu.min_chain_clusters) continue;
      ++cnt.starts;
      out.start_cluster.push_back(g);
      out.chain_len.push_back(len);
      const size_t tix = out.nhits.size();
      out.hits.resize((tix + 1) * R, -1);
      int32_t* hit = &out.hits[tix * R];

      // G15: initial state from the first two chain clusters.
      State st;
      {
        const uint32_t g1 = (uint32_t)o.up[g];
        const float dx = t.x[k0 + 1] - t.x[k0];
        const float m = (sc.Y(g1) - sc.Y(g)) / dx;
        const float q2 = std::sqrt(1.0f + m * m);
        st.y = sc.Y(g); st.z = sc.Z(g);
        st.s = m / q2;
        st.t = (sc.Z(g1) - sc.Z(g)) / (dx * q2);
        st.k = 0.0f;
        reset_cov(cu, st);
      }
      uint32_t cur = k0;
      hit[k0] = (int32_t)g;
      bool failed = false;
      State pr, nx; InvS w; float S00, S11;
      // ---- up pass, part 1: follow the chain, ungated (G22.1)
      for (int32_t c = o.up[g]; c >= 0; c = o.up[c]) {
        const uint32_t k = cur + 1;
        ++cnt.kf_row_steps;
        if (!transport(cu, st, t.x[k] - t.x[cur], 1.0f, pr) || !innovation(cu, pr, w, S00, S11) ||
            !update(cu, pr, w, sc.Y((uint32_t)c), sc.Z((uint32_t)c), nx)) { failed = true; break; }
        ++cnt.kf_updates;
        st = nx; cur = k; hit[k] = c;
      }
      // ---- up pass, part 2: extrapolate and pick up (G20, G21, G23)
      if (!failed) {
        uint32_t miss = 0;
        for (uint32_t k = cur + 1; k < R; ++k) {
          ++cnt.kf_row_steps;
          if (!transport(cu, st, t.x[k] - t.x[cur], (float)(k - cur), pr)) break;
          bool got = false;
          if (std::fabs(pr.y) <= t.ymax[k] + cu.edge_margin) {
            if (!innovation(cu, pr, w, S00, S11)) break;
            float c2;
            bool near = false;
            const int32_t b = best_on_row(sc, sc.rows[k], pr, w, S00, S11, c2, cnt, &near);
            if (near) { out.near.push_back((uint32_t)tix); out.near.push_back(k); }
            if (b >= 0) {
              if (!update(cu, pr, w, sc.Y((uint32_t)b), sc.Z((uint32_t)b), nx)) break;
              ++cnt.kf_updates;
              st = nx; cur = k; hit[k] = b; miss = 0; got = true;
            }
          }
          if (!got && ++miss > cu.max_row_gap) break;
        }
      }
      uint32_t last = cur;
      {
        const float tv[5] = {st.y, st.z, st.s, st.t, st.k};
        out.top.insert(out.top.end(), tv, tv + 5);
        out.top.insert(out.top.end(), st.c, st.c + 15);
      }
      // ---- down pass (G22.2): keep the state at the top hit row, reset C, refit downwards.
      reset_cov(cu, st);
      float chi2 = 0.f;
      uint32_t nh = 0;
      bool ok = innovation(cu, st, w, S00, S11);
      if (ok) {
        const uint32_t gt = (uint32_t)hit[last];
        chi2 = chi2 + chi2_of(w, sc.Y(gt) - st.y, sc.Z(gt) - st.z);
        ok = update(cu, st, w, sc.Y(gt), sc.Z(gt), nx);
      }
      if (ok) {
        ++cnt.kf_updates;
        st = nx; nh = 1;
        uint32_t miss = 0;
        for (int32_t k = (int32_t)last - 1; k >= 0; --k) {
          ++cnt.kf_row_steps;
          if (!transport(cu, st, t.x[k] - t.x[cur], (float)(cur - (uint32_t)k), pr)) break;
          const bool below = (uint32_t)k < k0;
          if (hit[k] >= 0) {                                   // existing hit: ungated refit
            if (!innovation(cu, pr, w, S00, S11)) break;
            const uint32_t gh = (uint32_t)hit[k];
            const float c2 = chi2_of(w, sc.Y(gh) - pr.y, sc.Z(gh) - pr.z);
            if (!update(cu, pr, w, sc.Y(gh), sc.Z(gh), nx)) break;
            ++cnt.kf_updates;
            chi2 = chi2 + c2; st = nx; cur = (uint32_t)k; ++nh;
            continue;
          }
          bool got = false;
          if (std::fabs(pr.y) <= t.ymax[k] + cu.edge_margin) {
            if (!innovation(cu, pr, w, S00, S11)) break;
            float c2;
            bool near = false;
            const int32_t b = best_on_row(sc, sc.rows[k], pr, w, S00, S11, c2, cnt, &near);
            if (near) { out.near.push_back((uint32_t)tix); out.near.push_back((uint32_t)k); }
            if (b >= 0) {
              if (!update(cu, pr, w, sc.Y((uint32_t)b), sc.Z((uint32_t)b), nx)) break;
              ++cnt.kf_updates;
              chi2 = chi2 + c2; st = nx; cur = (uint32_t)k; hit[k] = b; ++nh; got = true;
              if (below) miss = 0;
            }
          }
          if (!got && below && ++miss > cu.max_row_gap) break;
        }
      }
      // G22c (truncation rule): the tracklet spans [cur, last]; hits below cur (the down pass
      // failed inside the range: G16b / G24) are dropped.
      for (uint32_t k = 0; k < cur; ++k) hit[k] = -1;
      if (!ok) { nh = 0; }
      // G22d — further passes (NEXT-4; L45 "This is repeated until no more clusters are found"; cut
      // max_passes, default 2).  Pass 3 goes up again, pass 4 down, ...  A pass starts where the previous
      // one ended (the first row after a down pass, the top row after an up pass) from that state with the
      // covariance reset to the prior and chi2 = 0 (as G22.2), is updated with the hit of that row and
      // then walks to the other end and beyond: a row holding a hit -> ungated update; a row without ->
      // pickup (G20, G23), inside the range too; misses are counted beyond the far end of the range only
      // (G21), where a failure (G16b / G24) just ends the pass as it does in G21.  A pass that fails INSIDE
      // the range (it would shorten the tracklet) or picks up no NEW cluster is discarded and ends the
      // construction: the tracklet stays as the previous pass left it.  Otherwise the new clusters join the
      // tracklet, the range grows to the last update, nhits / chi2 / state are those of this pass, and the
      // state now sits at the row of its last update.
      uint32_t first = cur, ref = cur, passes = 2;
      for (uint32_t pass = 3; pass <= cu.max_passes && ok && nh > 0; ++pass) {
        const bool up = (pass & 1u) != 0u;
        const int32_t e = up ? (int32_t)first : (int32_t)last, dir = up ? 1 : -1;
        State s2 = st;
        reset_cov(cu, s2);
        float chi = 0.f;
        if (!innovation(cu, s2, w, S00, S11)) break;
        {
          const uint32_t ge = (uint32_t)hit[e];
          chi = chi + chi2_of(w, sc.Y(ge) - s2.y, sc.Z(ge) - s2.z);
          if (!update(cu, s2, w, sc.Y(ge), sc.Z(ge), nx)) break;
          ++cnt.kf_updates;
          s2 = nx;
        }
        std::vector<int32_t> nh2(hit, hit + R);
        uint32_t n2 = 1, gained = 0, miss = 0, c2row = (uint32_t)e;
        bool bad = false;
        for (int32_t k = e + dir; k >= 0 && k < (int32_t)R; k += dir) {
          ++cnt.kf_row_steps;
          const uint32_t nr = (uint32_t)k > c2row ? (uint32_t)k - c2row : c2row - (uint32_t)k;
          const bool beyond = up ? (uint32_t)k > last : (uint32_t)k < first;
          if (!transport(cu, s2, t.x[k] - t.x[c2row], (float)nr, pr)) { bad = !beyond; break; }
          int32_t g2 = nh2[k];
          float c2 = 0.f;
          if (g2 >= 0) {
            if (!innovation(cu, pr, w, S00, S11)) { bad = !beyond; break; }
            c2 = chi2_of(w, sc.Y((uint32_t)g2) - pr.y, sc.Z((uint32_t)g2) - pr.z);
          } else if (std::fabs(pr.y) <= t.ymax[k] + cu.edge_margin) {
            if (!innovation(cu, pr, w, S00, S11)) { bad = !beyond; break; }
            bool near = false;
            g2 = best_on_row(sc, sc.rows[k], pr, w, S00, S11, c2, cnt, &near);
            if (near) { out.near.push_back((uint32_t)tix); out.near.push_back((uint32_t)k); }
            if (g2 >= 0) { nh2[k] = g2; ++gained; }
          }
          if (g2 >= 0) {
            if (!update(cu, pr, w, sc.Y((uint32_t)g2), sc.Z((uint32_t)g2), nx)) { bad = !beyond; if (beyond) { nh2[k] = -1; --gained; } break; }
            ++cnt.kf_updates;
            chi = chi + c2; s2 = nx; c2row = (uint32_t)k; ++n2;
            if (beyond) miss = 0;
          } else if (beyond && ++miss > cu.max_row_gap) {
            break;
          }
        }
        if (bad || gained == 0) break;
        for (uint32_t k = 0; k < R; ++k) hit[k] = nh2[k];
        st = s2; chi2 = chi; nh = n2; passes = pass;
        if (up) last = c2row; else first = c2row;
        ref = c2row;
      }
      out.first_row.push_back(first);
      out.last_row.push_back(last);
      out.ref_row.push_back(ref);
      out.n_passes.push_back(passes);
      out.nhits.push_back(nh);
      out.chi2.push_back(chi2);
      const float pv[5] = {st.y, st.z, st.s, st.t, st.k};
      out.params.insert(out.params.end(), pv, pv + 5);
      out.cov.insert(out.cov.end(), st.c, st.c + 15);
    }
  }
}

// ---------------------------------------------------------------------------------------------
// Step 6 — selection (L46, L78, L116; G26).  key = (nhits << 24) | (0xFFFFFF - t_local); the
// owner of a cluster is the claimant with the maximal key.  select_mode 1 (NEXT-1, L80-L94):
// weight w = n * (alpha - chi2 / ndf) ranks the claimants instead of n.
inline uint32_t float_order_bits(float w) {                    // order-preserving map float -> uint32
  uint32_t b; std::memcpy(&b, &w, 4);
  return (b & 0x80000000u) ? ~b : (b | 0x80000000u);
}

// G26b (NEXT-4): with select_rounds = 2 the selection is repeated once among the tracklets the first
// round accepted: every owner of the sector is cleared, only accepted tracklets claim (same keys),
// kept counts and cuts are evaluated again.  A tracklet can only gain clusters in the second round
// (there are fewer claimants), so the accepted set is unchanged; what changes is that the clusters
// a rejected tracklet had won go to the accepted tracklet that also holds them, or become free.
void select_sector(Oracle& o, const SectorCtx& sc, SectorResult& out) {
  const uint32_t R = o.geo.n_rows;
  const Cuts& cu = o.cuts;
  const size_t T = out.nhits.size();
  out.kept.assign(T, 0); out.accepted.assign(T, 0);
  std::vector<uint32_t> key(T, 0);
  // mode 1 uses a 64-bit comparison (weight bits, then lower id); stored owner is the tracklet's
  // local id + 1 in that mode, the packed key in mode 0.
  std::vector<uint64_t> key64(T, 0);
  std::vector<uint64_t> best64;
  const uint32_t g_end = o.row_start[(sc.sector + 1) * R];
  for (uint32_t round = 0; round < (cu.select_rounds >= 2u ? 2u : 1u); ++round) {
    if (round > 0) for (uint32_t g = sc.g_base; g < g_end; ++g) o.owner[g] = 0u;
    if (cu.select_mode == 1) best64.assign(g_end - sc.g_base, 0);
    for (size_t ti = 0; ti < T; ++ti) {
      key[ti] = 0;
      if (out.nhits[ti] < cu.min_clusters) continue;             // G26: only these claim
      if (round > 0 && !out.accepted[ti]) continue;              // G26b: ... and in round 2 only the accepted ones
      if (cu.select_mode == 0) {
        key[ti] = (out.nhits[ti] << 24) | (0xFFFFFFu - (uint32_t)ti);
      } else {
        const float n = (float)out.nhits[ti];
        const float ndf = 2.0f * n - 5.0f;
        const float wgt = n * (cu.alpha - out.chi2[ti] / ndf);
        key64[ti] = ((uint64_t)float_order_bits(wgt) << 32) | (uint64_t)(0xFFFFFFFFu - (uint32_t)ti);
        key[ti] = (uint32_t)ti + 1u;
      }
      const int32_t* hit = &out.hits[ti * R];
      for (uint32_t k = out.first_row[ti]; k <= out.last_row[ti]; ++k) {
        if (hit[k] < 0) continue;
        if (round == 0) ++out.cnt.claimed_hits;
        if (cu.select_mode == 0) { if (key[ti] > o.owner[hit[k]]) o.owner[hit[k]] = key[ti]; }
        else if (key64[ti] > best64[hit[k] - sc.g_base]) { best64[hit[k] - sc.g_base] = key64[ti]; o.owner[hit[k]] = key[ti]; }
      }
    }
    for (size_t ti = 0; ti < T; ++ti) {
      if (key[ti] == 0) { out.kept[ti] = 0; out.accepted[ti] = 0; continue; }
      const int32_t* hit = &out.hits[ti * R];
      uint32_t kept = 0;
      for (uint32_t k = out.first_row[ti]; k <= out.last_row[ti]; ++k)
        if (hit[k] >= 0 && o.owner[hit[k]] == key[ti]) ++kept;
      out.kept[ti] = kept;
      const float qpt = (0.0f - out.params[ti * 5 + 4]) / o.tab.kbz;       // G14
      out.accepted[ti] = (kept >= cu.min_clusters && std::fabs(qpt) <= o.tab.max_qpt) ? 1 : 0;
    }
  }
}

void run_sector(Oracle& o, const float* xyz, uint32_t sector, int mode, int stop_after, SectorResult& out) {
  SectorCtx sc; sc.o = &o; sc.xyz = xyz; sc.sector = sector; sc.mode = mode;
  bin_sector(o, sc);
  if (stop_after == 1) return;
  neighbours_sector(o, sc, out.cnt);
  evolve_sector(o, sc, out.cnt);
  if (stop_after == 3) return;
  construct_sector(o, sc, out);
  select_sector(o, sc, out);
}

// ---------------------------------------------------------------------------------------------
// NEXT-2 — global tracking (section 5; readings G33-G36 of DESIGN.md).
// "Having finished the sector tracking the tracker searches for track segments ending in the
// innermost or outermost part of the TPC at the edge of a sector.  The track parameters are then
// converted to the coordinate system of the neighboring sectors and the tracklet construction step
// is continued."  The paper gives no number, formula or rule beyond these two sentences.
//
// G34: rotation of the state at x0 into the frame of the neighbour on the side of sg = sign(y)
// (frames differ by the angle dphi = 2 atan(tan_half_angle); local y grows with azimuth):
//   x' = x0*cd + y*sds,  y' = y*cd - x0*sds,  sin phi' = s*cd - c*sds   (c = sqrt(1 - s*s), sds = sg*sd)
// z, dz/ds and kappa are unchanged.  Covariance: C'ij = (Ji*Cij)*Jj with J = (c/c', 1, c'/c, 1, 1)
// (the couplings d s'/d y = -kappa sds and d z'/d y = -t sds/c' are neglected, as d z'/d s is in G16).
bool rotate_state(const Cuts& cu, const Tables& t, const State& a, float x0, float sg, State& b, float& xr) {
  const float cd = t.gt_cos, sds = sg * t.gt_sin;
  xr = x0 * cd + a.y * sds;
  b.y = a.y * cd - x0 * sds;
  const float c = std::sqrt(1.0f - a.s * a.s);
  b.s = a.s * cd - c * sds;
  if (!(std::fabs(b.s) <= cu.max_sinphi)) return false;
  const float c1 = std::sqrt(1.0f - b.s * b.s);
  b.z = a.z; b.t = a.t; b.k = a.k;
  const float J[5] = {c / c1, 1.0f, c1 / c, 1.0f, 1.0f};
  for (int i = 0; i < 5; ++i)
    for (int j = 0; j <= i; ++j) C(b, i, j) = (J[i] * Cc(a, i, j)) * J[j];
  return true;
}

// G33, G35, G36.  For every output track and each of its two ends: the end qualifies if at most
// gt_max_rows rows lie beyond it (the piece in the neighbour is then too short to be a sector track,
// L116) and the state there lies within gt_edge of the sector edge.  Inner end: the track parameters
// (state at first_row after the down pass); outer end: the state at the top hit row at the end of
// the up pass.  The state is rotated (G34) and the construction continues row by row away from the
// segment in the neighbour: transport from the last update, outside-of-sector = miss (G23), pickup
// (G20) among the FREE clusters of the row (owner == 0: claimed by no tracklet of >= min_clusters
// hits), update, until misses > max_row_gap, a failure, or the last row.  One hop only; two
// prolongations may pick up the same free cluster (no second selection).  Plain definition: the
// pickup scans the whole row.
void global_tracking(Oracle& o, const float* xyz, const std::vector<State>& low, const std::vector<State>& top) {
  const Cuts& cu = o.cuts; const Tables& t = o.tab;
  const uint32_t R = o.geo.n_rows, S = o.geo.n_sectors;
  if (S % 18u != 0u) return;                                    // needs the full ring of sectors
  for (size_t ti = 0; ti < o.tracks.size(); ++ti) {
    const Track& tk = o.tracks[ti];
    for (uint32_t end = 0; end < 2; ++end) {
      const uint32_t kend = end == 0 ? tk.first_row : tk.last_row;
      const uint32_t beyond = end == 0 ? kend : R - 1u - kend;
      if (beyond == 0u || beyond > cu.gt_max_rows) continue;
      const State& a = end == 0 ? low[ti] : top[ti];
      if (!(std::fabs(a.y) >= t.ymax[kend] - cu.gt_edge)) continue;
      const float sg = a.y >= 0.0f ? 1.0f : -1.0f;
      const uint32_t half = tk.sector / 18u, j = tk.sector % 18u;
      const uint32_t nb = half * 18u + (sg > 0.0f ? (j + 1u) % 18u : (j + 17u) % 18u);
      State st, pr, nx; float xcur;
      if (!rotate_state(cu, t, a, t.x[kend], sg, st, xcur)) continue;
      GlobalExt ge; std::memset(&ge, 0, sizeof(ge));
      ge.track = (uint32_t)ti; ge.sector = nb; ge.end = end; ge.first_cluster = (uint32_t)o.global_cluster_ids.size();
      uint32_t miss = 0, kref = kend; float chi2 = 0.0f;
      for (int32_t k = end == 0 ? (int32_t)kend - 1 : (int32_t)kend + 1; k >= 0 && k < (int32_t)R; k += end == 0 ? -1 : 1) {
        const uint32_t nr = (uint32_t)k > kref ? (uint32_t)k - kref : kref - (uint32_t)k;
        if (!transport(cu, st, t.x[k] - xcur, (float)nr, pr)) break;
        bool got = false;
        if (std::fabs(pr.y) <= t.ymax[k] + cu.edge_margin) {
          InvS w; float S00, S11;
          if (!innovation(cu, pr, w, S00, S11)) break;
          int64_t best = -1; float best_c2 = 0.0f;
          const uint32_t sr = nb * R + (uint32_t)k;
          for (uint32_t g = o.row_start[sr]; g < o.row_start[sr + 1]; ++g) {
            if (o.owner[g] != 0u) continue;
            const float c2 = chi2_of(w, xyz[3 * (size_t)g + 1] - pr.y, xyz[3 * (size_t)g + 2] - pr.z);
            if (!(c2 <= cu.chi2_cut)) continue;
            if (best < 0 || c2 < best_c2) { best = g; best_c2 = c2; }     // g ascending: ties keep the smaller index
          }
          if (best >= 0) {
            if (!update(cu, pr, w, xyz[3 * (size_t)best + 1], xyz[3 * (size_t)best + 2], nx)) break;
            st = nx; xcur = t.x[k]; kref = (uint32_t)k; miss = 0; got = true; chi2 = chi2 + best_c2;
            o.global_cluster_ids.push_back((uint32_t)best);
            ++ge.n_clusters; ge.row = (uint32_t)k;
          }
        }
        if (!got && ++miss > cu.max_row_gap) break;
      }
      if (ge.n_clusters == 0u) continue;
      ge.x_ref = t.x[ge.row]; ge.y = st.y; ge.z = st.z; ge.sinphi = st.s; ge.dzds = st.t;
      ge.qpt = (0.0f - st.k) / t.kbz;
      std::memcpy(ge.cov, st.c, sizeof(ge.cov)); ge.chi2 = chi2;
      o.global_ext.push_back(ge);
    }
  }
}

template <class T> void append(std::vector<T>& a, const std::vector<T>& b) { a.insert(a.end(), b.begin(), b.end()); }

}  // namespace

// ---------------------------------------------------------------------------------------------
// C interface for ctypes (oracle/oracle.py).
// ---------------------------------------------------------------------------------------------
// NEXT-3 — track sort, refit and merging of sector tracks ("the sector tracks are merged
// by the track merger", L98 "a fast sorting of the tracks in between of sector tracking and track
// merging", L102 "[the sector tracker] outputs a list of clusters for each track and the track merger
// does a refit of the track"; readings G37-G40 of DESIGN.md).  The paper says no more than these
// sentences.  Only the cluster lists and the row ranges of the sector tracks are used: none of the
// sector tracker's intermediate floating-point results enters (L102).
//   G37 sort: canonical order of the tracks = ascending (sector, first_row, seed_cluster).
//   G38 refit: outward pass over the list (state from the first two clusters as in G15, then
//       transport + ungated update cluster by cluster) -> state at the last row; inward pass as the
//       down pass of G22.2 (covariance reset, update with the top cluster, then down the list) -> state
//       at the first row, chi2 = sum of the inward increments.  Any failure: ok = 0, record zeroed.
//   G39 match: segment A may be continued by B if B lies in the neighbouring sector on the side of
//       sign(y) of A's outer state, 1 <= row_in(B) - row_out(A) <= merge_max_gap (rows of B's first and
//       of A's last cluster) and both are ok.
//       A's outer state is rotated into B's frame (G34), transported to x[row_in(B)] over that many
//       rows; chi2 = sum over the 5 parameters of d_i^2 / (C_ii(A') + C_ii(B inner)), left to right;
//       accepted iff chi2 <= merge_chi2_cut.
//   G40 links: for A the accepted B of minimal chi2, for B the accepted A of minimal chi2 (ties ->
//       lower rank); a link is kept iff the two agree (the rule of the evolution step, L41).
//   G41 merged track = chain of segments through `next`, reported at its first segment: a chain of one
//       segment repeats that segment's refit; a longer chain is refitted jointly (L102) as in G38 over
//       the concatenated cluster lists, the state being rotated (G34) into the next segment's frame after
//       the last cluster of a segment on the way out, and back on the way in; the first transport after
//       a rotation starts at the rotated x and counts the rows between the two clusters.
void merge_sector_tracks(Oracle& o, const float* xyz) {
  const Cuts& cu = o.cuts; const Tables& t = o.tab;
  const uint32_t R = o.geo.n_rows, S = o.geo.n_sectors;
  const size_t K = o.tracks.size();
  MergeSeg zero; std::memset(&zero, 0, sizeof(zero)); zero.next = zero.prev = -1;
  o.merge.assign(K, zero);
  o.merge_cand.clear();
  // G37
  std::vector<uint32_t> order(K);
  for (size_t i = 0; i < K; ++i) order[i] = (uint32_t)i;
  std::sort(order.begin(), order.end(), [&](uint32_t a, uint32_t b) {
    const Track &x = o.tracks[a], &y = o.tracks[b];
    if (x.sector != y.sector) return x.sector < y.sector;
    if (x.first_row != y.first_row) return x.first_row < y.first_row;
    return x.seed_cluster < y.seed_cluster;
  });
  for (size_t i = 0; i < K; ++i) o.merge[order[i]].rank = (uint32_t)i;
  // G38
  std::vector<State> inner(K), outer(K);
  for (size_t ti = 0; ti < K; ++ti) {
    const Track& tk = o.tracks[ti];
    MergeSeg& m = o.merge[ti];
    const uint32_t n = tk.n_clusters;
    if (n < 2u) continue;
    const uint32_t* ids = &o.track_cluster_ids[tk.first_cluster];
    std::vector<uint32_t> row(n);
    for (uint32_t i = 0; i < n; ++i) {                           // row of a cluster from the caller's row_start
      uint32_t k = 0;
      while (!(o.row_start[tk.sector * R + k] <= ids[i] && ids[i] < o.row_start[tk.sector * R + k + 1])) ++k;
      row[i] = k;
    }
    auto Y = [&](uint32_t i) { return xyz[3 * (size_t)ids[i] + 1]; };
    auto Z = [&](uint32_t i) { return xyz[3 * (size_t)ids[i] + 2]; };
    State st, pr, nx; InvS w; float S00, S11;
    {
      const float dx = t.x[row[1]] - t.x[row[0]];
      const float mm = (Y(1) - Y(0)) / dx;
      const float q2 = std::sqrt(1.0f + mm * mm);
      st.y = Y(0); st.z = Z(0);
      st.s = mm / q2;
      st.t = (Z(1) - Z(0)) / (dx * q2);
      st.k = 0.0f;
      reset_cov(cu, st);
    }
    bool ok = true;
    uint32_t cur = row[0];
    for (uint32_t i = 1; i < n && ok; ++i) {
      ok = transport(cu, st, t.x[row[i]] - t.x[cur], (float)(row[i] - cur), pr) && innovation(cu, pr, w, S00, S11) &&
           update(cu, pr, w, Y(i), Z(i), nx);
      if (ok) { st = nx; cur = row[i]; }
    }
    if (!ok) continue;
    outer[ti] = st;
    reset_cov(cu, st);
    float chi2 = 0.0f;
    ok = innovation(cu, st, w, S00, S11);
    if (ok) {
      chi2 = chi2 + chi2_of(w, Y(n - 1) - st.y, Z(n - 1) - st.z);
      ok = update(cu, st, w, Y(n - 1), Z(n - 1), nx);
    }
    if (ok) st = nx;
    for (int32_t i = (int32_t)n - 2; i >= 0 && ok; --i) {
      ok = transport(cu, st, t.x[row[i]] - t.x[cur], (float)(cur - row[i]), pr) && innovation(cu, pr, w, S00, S11);
      if (!ok) break;
      const float c2 = chi2_of(w, Y((uint32_t)i) - pr.y, Z((uint32_t)i) - pr.z);
      ok = update(cu, pr, w, Y((uint32_t)i), Z((uint32_t)i), nx);
      if (ok) { chi2 = chi2 + c2; st = nx; cur = row[i]; }
    }
    if (!ok) continue;
    inner[ti] = st;
    m.ok = 1u; m.chi2 = chi2; m.row_in = row[0]; m.row_out = row[n - 1];
    const float pi[5] = {st.y, st.z, st.s, st.t, st.k}, po[5] = {outer[ti].y, outer[ti].z, outer[ti].s, outer[ti].t, outer[ti].k};
    std::memcpy(m.in_par, pi, sizeof(pi)); std::memcpy(m.in_cov, st.c, sizeof(st.c));
    std::memcpy(m.out_par, po, sizeof(po)); std::memcpy(m.out_cov, outer[ti].c, sizeof(st.c));
  }
  // G39, G40 (matching needs the full ring of sectors; without it every track is a chain of one, G41)
  std::vector<int64_t> bestB(K, -1), bestA(K, -1);
  std::vector<float> chiB(K, 0.0f), chiA(K, 0.0f);
  for (size_t a = 0; a < K && S % 18u == 0u; ++a) {
    if (!o.merge[a].ok) continue;
    const Track& ta = o.tracks[a];
    const State& sa = outer[a];
    const float sg = sa.y >= 0.0f ? 1.0f : -1.0f;
    const uint32_t half = ta.sector / 18u, j = ta.sector % 18u;
    const uint32_t nb = half * 18u + (sg > 0.0f ? (j + 1u) % 18u : (j + 17u) % 18u);
    State rot, pr; float xr;
    const uint32_t ra = o.merge[a].row_out;
    if (!rotate_state(cu, t, sa, t.x[ra], sg, rot, xr)) continue;
    for (size_t b = 0; b < K; ++b) {
      const Track& tb = o.tracks[b];
      if (tb.sector != nb || !o.merge[b].ok) continue;
      const uint32_t rb = o.merge[b].row_in;
      if (!(rb > ra && rb - ra <= cu.merge_max_gap)) continue;
      if (!transport(cu, rot, t.x[rb] - xr, (float)(rb - ra), pr)) continue;
      const State& sb = inner[b];
      const float d[5] = {pr.y - sb.y, pr.z - sb.z, pr.s - sb.s, pr.t - sb.t, pr.k - sb.k};
      float chi2 = 0.0f;
      bool good = true;
      for (int i = 0; i < 5; ++i) {
        const float v = Cc(pr, i, i) + Cc(sb, i, i);
        if (!(v > 0.0f)) { good = false; break; }
        chi2 = chi2 + (d[i] * d[i]) / v;
      }
      if (!good || !(chi2 <= cu.merge_chi2_cut)) continue;
      o.merge_cand.push_back(MergeCand{(uint32_t)a, (uint32_t)b, chi2});
      if (bestB[a] < 0 || chi2 < chiB[a] || (chi2 == chiB[a] && o.merge[b].rank < o.merge[bestB[a]].rank)) { bestB[a] = (int64_t)b; chiB[a] = chi2; }
      if (bestA[b] < 0 || chi2 < chiA[b] || (chi2 == chiA[b] && o.merge[a].rank < o.merge[bestA[b]].rank)) { bestA[b] = (int64_t)a; chiA[b] = chi2; }
    }
  }
  for (size_t a = 0; a < K; ++a) {
    const int64_t b = bestB[a];
    if (b >= 0 && bestA[(size_t)b] == (int64_t)a) {
      o.merge[a].next = (int32_t)b; o.merge[a].match_chi2 = chiB[a];
      o.merge[(size_t)b].prev = (int32_t)a;
    }
  }
  // G41
  for (size_t h = 0; h < K; ++h) {
    MergeSeg& m = o.merge[h];
    if (m.prev >= 0 || !m.ok) continue;
    if (m.next < 0) {                                           // a chain of one segment: its own refit
      m.chain_n_seg = 1; m.chain_n_clusters = o.tracks[h].n_clusters; m.chain_chi2 = m.chi2;
      std::memcpy(m.chain_par, m.in_par, sizeof(m.in_par)); std::memcpy(m.chain_cov, m.in_cov, sizeof(m.in_cov));
      continue;
    }
    // concatenated list: (segment, cluster id, row) in the order of the outward pass
    struct Hit { uint32_t seg, id, row; };
    std::vector<Hit> hits;
    std::vector<uint32_t> segs;
    for (int32_t sgi = (int32_t)h; sgi >= 0; sgi = o.merge[(size_t)sgi].next) {
      const Track& tk = o.tracks[(size_t)sgi];
      segs.push_back((uint32_t)sgi);
      for (uint32_t i = 0; i < tk.n_clusters; ++i) {
        const uint32_t id = o.track_cluster_ids[tk.first_cluster + i];
        uint32_t k = 0;
        while (!(o.row_start[tk.sector * R + k] <= id && id < o.row_start[tk.sector * R + k + 1])) ++k;
        hits.push_back(Hit{(uint32_t)(segs.size() - 1), id, k});
      }
    }
    auto Y = [&](size_t i) { return xyz[3 * (size_t)hits[i].id + 1]; };
    auto Z = [&](size_t i) { return xyz[3 * (size_t)hits[i].id + 2]; };
    auto side = [&](uint32_t from, uint32_t to) {                // +1: `to` is the next sector in azimuth
      return ((o.tracks[segs[to]].sector + 18u - o.tracks[segs[from]].sector) % 18u) == 1u ? 1.0f : -1.0f;
    };
    const size_t n = hits.size();
    State st, pr, nx, rot; InvS w; float S00, S11;
    {
      const float dx = t.x[hits[1].row] - t.x[hits[0].row];
      const float mm = (Y(1) - Y(0)) / dx;
      const float q2 = std::sqrt(1.0f + mm * mm);
      st.y = Y(0); st.z = Z(0); st.s = mm / q2; st.t = (Z(1) - Z(0)) / (dx * q2); st.k = 0.0f;
      reset_cov(cu, st);
    }
    bool ok = true;
    float xcur = t.x[hits[0].row];
    for (size_t i = 1; i < n && ok; ++i) {
      if (hits[i].seg != hits[i - 1].seg) {                      // into the next segment's frame
        ok = rotate_state(cu, t, st, xcur, side(hits[i - 1].seg, hits[i].seg), rot, xcur);
        if (!ok) break;
        st = rot;
      }
      ok = transport(cu, st, t.x[hits[i].row] - xcur, (float)(hits[i].row - hits[i - 1].row), pr) && innovation(cu, pr, w, S00, S11) &&
           update(cu, pr, w, Y(i), Z(i), nx);
      if (ok) { st = nx; xcur = t.x[hits[i].row]; }
    }
    if (!ok) continue;
    reset_cov(cu, st);
    float chi2 = 0.0f;
    ok = innovation(cu, st, w, S00, S11);
    if (ok) {
      chi2 = chi2 + chi2_of(w, Y(n - 1) - st.y, Z(n - 1) - st.z);
      ok = update(cu, st, w, Y(n - 1), Z(n - 1), nx);
    }
    if (ok) st = nx;
    for (int64_t i = (int64_t)n - 2; i >= 0 && ok; --i) {
      if (hits[(size_t)i].seg != hits[(size_t)i + 1].seg) {      // back into the previous segment's frame
        ok = rotate_state(cu, t, st, xcur, -side(hits[(size_t)i].seg, hits[(size_t)i + 1].seg), rot, xcur);
        if (!ok) break;
        st = rot;
      }
      ok = transport(cu, st, t.x[hits[(size_t)i].row] - xcur, (float)(hits[(size_t)i + 1].row - hits[(size_t)i].row), pr) &&
           innovation(cu, pr, w, S00, S11);
      if (!ok) break;
      const float c2 = chi2_of(w, Y((size_t)i) - pr.y, Z((size_t)i) - pr.z);
      ok = update(cu, pr, w, Y((size_t)i), Z((size_t)i), nx);
      if (ok) { chi2 = chi2 + c2; st = nx; xcur = t.x[hits[(size_t)i].row]; }
    }
    if (!ok) continue;
    m.chain_n_seg = (uint32_t)segs.size(); m.chain_n_clusters = (uint32_t)n; m.chain_chi2 = chi2;
    const float pc[5] = {st.y, st.z, st.s, st.t, st.k};
    std::memcpy(m.chain_par, pc, sizeof(pc)); std::memcpy(m.chain_cov, st.c, sizeof(st.c));
  }
}

extern "C" {

void* orc_create(const Geometry* g, const Cuts* c) {
  Oracle* o = new Oracle();
  o->geo = *g;
  o->row_x.assign(g->row_x, g->row_x + g->n_rows);
  o->geo.row_x = o->row_x.data();
  o->cuts = *c;
  build_tables(*o);
  return o;
}
void orc_destroy(void* h) { delete (Oracle*)h; }

// Run the tracker on one event.  mode: 0 grid, 1 row scan, 2 all triplets (neighbours finder).
// stop_after: 0 = all steps, 1 = after binning, 3 = after evolution.  n_threads: sectors are
// independent (L28, L112 "trivial parallelization over the sectors"); 1 = single thread.
int orc_run(void* h, const float* xyz, const uint32_t* row_start, uint32_t n, int mode, int stop_after, int n_threads) {
  Oracle& o = *(Oracle*)h;
  const uint32_t S = o.geo.n_sectors, R = o.geo.n_rows;
  o.n = n;
  o.row_start.assign(row_start, row_start + S * R + 1);
  if (o.row_start[S * R] != n) return -1;
  for (uint32_t i = 0; i < S * R; ++i) if (o.row_start[i] > o.row_start[i + 1]) return -1;
  o.bin_row_offset.assign(S * R + 1, 0);
  for (uint32_t sr = 0; sr < S * R; ++sr) o.bin_row_offset[sr + 1] = o.bin_row_offset[sr] + o.tab.ny[sr % R] * o.tab.nz;
  o.bin_of.assign(n, 0);
  o.bin_count.assign(o.bin_row_offset[S * R], 0); o.bin_start.assign(o.bin_row_offset[S * R], 0);
  o.up_raw.assign(n, -1); o.dn_raw.assign(n, -1); o.up.assign(n, -1); o.dn.assign(n, -1);
  o.owner.assign(n, 0);
  std::vector<SectorResult> res(S);
  if (n_threads <= 1) {
    for (uint32_t s = 0; s < S; ++s) run_sector(o, xyz, s, mode, stop_after, res[s]);
  } else {
    std::atomic<uint32_t> next{0};
    std::vector<std::thread> th;
    for (int i = 0; i < n_threads; ++i)
      th.emplace_back([&]() { for (uint32_t s; (s = next.fetch_add(1)) < S;) run_sector(o, xyz, s, mode, stop_after, res[s]); });
    for (auto& x : th) x.join();
  }
  // Step 7 — output (L52, L102; G27, G28): tracklet ids in (sector, start row, original index)
  // order; surviving tracklets in id order; cluster lists in ascending row order; no refit.
  o.start_cluster.clear(); o.chain_len.clear(); o.first_row.clear(); o.last_row.clear(); o.nhits.clear();
  o.ref_row.clear(); o.n_passes.clear(); o.near.clear();
  o.kept.clear(); o.accepted.clear(); o.params.clear(); o.cov.clear(); o.chi2.clear(); o.hits.clear();
  o.tracklet_sector.clear(); o.tracks.clear(); o.track_cluster_ids.clear();
  o.global_ext.clear(); o.global_cluster_ids.clear();
  std::vector<State> low, top;                       // NEXT-2: the two end states of every output track
  o.cnt = Counters();
  for (uint32_t s = 0; s < S; ++s) {
    SectorResult& r = res[s];
    const size_t T = r.nhits.size();
    for (size_t ti = 0; ti < T; ++ti) {
      if (!r.accepted.empty() && r.accepted[ti]) {
        Track tk;
        tk.sector = s; tk.first_row = r.first_row[ti]; tk.last_row = r.last_row[ti];
        tk.n_clusters = r.kept[ti]; tk.first_cluster = (uint32_t)o.track_cluster_ids.size();
        tk.seed_cluster = r.start_cluster[ti];
        tk.x_ref = o.tab.x[r.ref_row[ti]];                 // first_row unless an upward pass > 2 shaped the tracklet (G22d)
        tk.y = r.params[ti * 5]; tk.z = r.params[ti * 5 + 1]; tk.sinphi = r.params[ti * 5 + 2]; tk.dzds = r.params[ti * 5 + 3];
        tk.qpt = (0.0f - r.params[ti * 5 + 4]) / o.tab.kbz;
        std::memcpy(tk.cov, &r.cov[ti * 15], sizeof(tk.cov));
        tk.chi2 = r.chi2[ti];
        const uint32_t key = o.cuts.select_mode == 0 ? ((r.nhits[ti] << 24) | (0xFFFFFFu - (uint32_t)ti)) : (uint32_t)ti + 1u;
        for (uint32_t k = tk.first_row; k <= tk.last_row; ++k) {
          const int32_t hgl = r.hits[ti * R + k];
          if (hgl >= 0 && o.owner[hgl] == key) o.track_cluster_ids.push_back((uint32_t)hgl);
        }
        o.tracks.push_back(tk);
        State a;
        a.y = r.params[ti * 5]; a.z = r.params[ti * 5 + 1]; a.s = r.params[ti * 5 + 2]; a.t = r.params[ti * 5 + 3];
        a.k = r.params[ti * 5 + 4]; std::memcpy(a.c, &r.cov[ti * 15], sizeof(a.c));
        low.push_back(a);
        const float* tv = &r.top[ti * 20];
        a.y = tv[0]; a.z = tv[1]; a.s = tv[2]; a.t = tv[3]; a.k = tv[4]; std::memcpy(a.c, tv + 5, sizeof(a.c));
        top.push_back(a);
      }
    }
    append(o.start_cluster, r.start_cluster); append(o.chain_len, r.chain_len);
    append(o.first_row, r.first_row); append(o.last_row, r.last_row); append(o.nhits, r.nhits);
    for (size_t i = 0; i + 1 < r.near.size(); i += 2) { o.near.push_back((uint32_t)(o.nhits.size() - T) + r.near[i]); o.near.push_back(r.near[i + 1]); }
    append(o.ref_row, r.ref_row); append(o.n_passes, r.n_passes);
    append(o.kept, r.kept); append(o.accepted, r.accepted);
    append(o.params, r.params); append(o.cov, r.cov); append(o.chi2, r.chi2); append(o.hits, r.hits);
    o.tracklet_sector.insert(o.tracklet_sector.end(), T, s);
    const uint64_t* a = (const uint64_t*)&r.cnt; uint64_t* b = (uint64_t*)&o.cnt;
    for (size_t i = 0; i < sizeof(Counters) / 8; ++i) b[i] += a[i];
  }
  o.cnt.tracks = o.tracks.size(); o.cnt.track_clusters = o.track_cluster_ids.size();
  if (stop_after == 0 && o.cuts.global_tracking) global_tracking(o, xyz, low, top);
  o.merge.clear(); o.merge_cand.clear();
  if (stop_after == 0 && o.cuts.merge_tracks) merge_sector_tracks(o, xyz);
  return 0;
}

// Array access: returns a pointer into the oracle's storage and the element count.
enum { A_BIN_OF = 0, A_BIN_ROW_OFFSET, A_BIN_COUNT, A_BIN_START, A_UP_RAW, A_DN_RAW, A_UP, A_DN, A_OWNER,
       A_START_CLUSTER, A_CHAIN_LEN, A_FIRST_ROW, A_LAST_ROW, A_NHITS, A_KEPT, A_ACCEPTED, A_PARAMS, A_COV,
       A_CHI2, A_HITS, A_TRACKS, A_TRACK_CLUSTER_IDS, A_COUNTERS, A_TRACKLET_SECTOR,
       A_TAB_YMAX, A_TAB_NY, A_TAB_RATIO_UP, A_TAB_RATIO_DN, A_TAB_W_UP, A_TAB_W_DN,
       A_TAB_WY_UP, A_TAB_WY_DN, A_TAB_WZ_UP, A_TAB_WZ_DN, A_GLOBAL_EXT, A_GLOBAL_CLUSTER_IDS, A_MERGE, A_MERGE_CAND, A_REF_ROW, A_N_PASSES, A_NEAR };
const void* orc_array(void* h, int what, uint64_t* count) {
  Oracle& o = *(Oracle*)h;
#define RET(v) do { *count = (v).size(); return (v).data(); } while (0)
  switch (what) {
    case A_BIN_OF: RET(o.bin_of); case A_BIN_ROW_OFFSET: RET(o.bin_row_offset);
    case A_BIN_COUNT: RET(o.bin_count); case A_BIN_START: RET(o.bin_start);
    case A_UP_RAW: RET(o.up_raw); case A_DN_RAW: RET(o.dn_raw); case A_UP: RET(o.up); case A_DN: RET(o.dn);
    case A_OWNER: RET(o.owner); case A_START_CLUSTER: RET(o.start_cluster); case A_CHAIN_LEN: RET(o.chain_len);
    case A_FIRST_ROW: RET(o.first_row); case A_LAST_ROW: RET(o.last_row); case A_NHITS: RET(o.nhits);
    case A_KEPT: RET(o.kept); case A_ACCEPTED: RET(o.accepted); case A_PARAMS: RET(o.params); case A_COV: RET(o.cov);
    case A_CHI2: RET(o.chi2); case A_HITS: RET(o.hits); case A_TRACKS: RET(o.tracks);
    case A_TRACK_CLUSTER_IDS: RET(o.track_cluster_ids); case A_TRACKLET_SECTOR: RET(o.tracklet_sector);
    case A_COUNTERS: *count = sizeof(Counters) / 8; return &o.cnt;
    case A_TAB_YMAX: RET(o.tab.ymax); case A_TAB_NY: RET(o.tab.ny);
    case A_TAB_RATIO_UP: RET(o.tab.ratio_up); case A_TAB_RATIO_DN: RET(o.tab.ratio_dn);
    case A_TAB_W_UP: RET(o.tab.w_up); case A_TAB_W_DN: RET(o.tab.w_dn);
    case A_TAB_WY_UP: RET(o.tab.wy_up); case A_TAB_WY_DN: RET(o.tab.wy_dn);
    case A_TAB_WZ_UP: RET(o.tab.wz_up); case A_TAB_WZ_DN: RET(o.tab.wz_dn);
    case A_GLOBAL_EXT: RET(o.global_ext); case A_GLOBAL_CLUSTER_IDS: RET(o.global_cluster_ids);
    case A_MERGE: RET(o.merge); case A_MERGE_CAND: RET(o.merge_cand);
    case A_REF_ROW: RET(o.ref_row); case A_N_PASSES: RET(o.n_passes); case A_NEAR: RET(o.near);
  }
#undef RET
  *count = 0; return nullptr;
}
uint32_t orc_nz(void* h) { return ((Oracle*)h)->tab.nz; }

// Single-step entry points used by the closed-form pins (tests/test_oracle_kalman.py).
// state = (y, z, s, t, k) + 15 covariance elements (lower triangle, row-major).
int orc_transport(void* h, const float* in20, float dx, float nrows, float* out20) {
  Oracle& o = *(Oracle*)h; State a, b;
  a.y = in20[0]; a.z = in20[1]; a.s = in20[2]; a.t = in20[3]; a.k = in20[4]; std::memcpy(a.c, in20 + 5, 60);
  if (!transport(o.cuts, a, dx, nrows, b)) return 0;
  out20[0] = b.y; out20[1] = b.z; out20[2] = b.s; out20[3] = b.t; out20[4] = b.k; std::memcpy(out20 + 5, b.c, 60);
  return 1;
}
int orc_update(void* h, const float* in20, float ym, float zm, float* out20, float* chi2) {
  Oracle& o = *(Oracle*)h; State a, b; InvS w; float S00, S11;
  a.y = in20[0]; a.z = in20[1]; a.s = in20[2]; a.t = in20[3]; a.k = in20[4]; std::memcpy(a.c, in20 + 5, 60);
  if (!innovation(o.cuts, a, w, S00, S11)) return 0;
  *chi2 = chi2_of(w, ym - a.y, zm - a.z);
  if (!update(o.cuts, a, w, ym, zm, b)) return 0;
  out20[0] = b.y; out20[1] = b.z; out20[2] = b.s; out20[3] = b.t; out20[4] = b.k; std::memcpy(out20 + 5, b.c, 60);
  return 1;
}

// G34 rotation alone (pins): sg = +1 / -1, x0 = x of the state; returns 0 if it fails.
int orc_rotate(void* h, const float* in20, float x0, float sg, float* out20, float* xr) {
  Oracle& o = *(Oracle*)h; State a, b;
  a.y = in20[0]; a.z = in20[1]; a.s = in20[2]; a.t = in20[3]; a.k = in20[4]; std::memcpy(a.c, in20 + 5, 60);
  if (!rotate_state(o.cuts, o.tab, a, x0, sg, b, *xr)) return 0;
  out20[0] = b.y; out20[1] = b.z; out20[2] = b.s; out20[3] = b.t; out20[4] = b.k; std::memcpy(out20 + 5, b.c, 60);
  return 1;
}

// Diagnostic for the rest of NEXT-4 ("... until no more clusters are found"; G22 stops
// after the up and the down pass): what a THIRD pass would add.  For every tracklet of the last orc_run the
// pass is simulated without touching the results: state of the tracklet at its first row, covariance reset
// to the prior (as at the start of the down pass), update with the bottom hit, then upwards row by row:
// a row holding a hit -> ungated update; otherwise pickup (G20, whole row scanned) -> a cluster that would
// be NEW; misses count above the top hit row only.  gained[t] = number of new clusters, with bit 31 set if the
// simulated pass ended on a failure (G16b / G24; G22d discards such a pass).  Returns the sum of the new clusters.
uint64_t orc_third_pass_gain(void* h, const float* xyz, uint32_t* gained) {
  Oracle& o = *(Oracle*)h;
  const Cuts& cu = o.cuts; const Tables& t = o.tab;
  const uint32_t R = o.geo.n_rows;
  uint64_t total = 0;
  for (size_t ti = 0; ti < o.nhits.size(); ++ti) {
    gained[ti] = 0;
    if (o.nhits[ti] == 0) continue;
    const int32_t* hit = &o.hits[ti * R];
    const uint32_t sector = o.tracklet_sector[ti], first = o.first_row[ti], last = o.last_row[ti];
    State st, pr, nx; InvS w; float S00, S11;
    st.y = o.params[ti * 5]; st.z = o.params[ti * 5 + 1]; st.s = o.params[ti * 5 + 2]; st.t = o.params[ti * 5 + 3]; st.k = o.params[ti * 5 + 4];
    reset_cov(cu, st);
    if (hit[first] < 0 || !innovation(cu, st, w, S00, S11)) continue;
    if (!update(cu, st, w, xyz[3 * (size_t)hit[first] + 1], xyz[3 * (size_t)hit[first] + 2], nx)) continue;
    st = nx;
    uint32_t cur = first, miss = 0;
    for (uint32_t k = first + 1; k < R; ++k) {
      if (!transport(cu, st, t.x[k] - t.x[cur], (float)(k - cur), pr)) { if (k <= last) gained[ti] |= 0x80000000u; break; }
      int64_t g = k <= last ? hit[k] : -1;
      bool is_new = false;
      if (g < 0 && std::fabs(pr.y) <= t.ymax[k] + cu.edge_margin) {
        if (!innovation(cu, pr, w, S00, S11)) { if (k <= last) gained[ti] |= 0x80000000u; break; }
        float best = 0.0f;
        const uint32_t sr = sector * R + k;
        for (uint32_t q = o.row_start[sr]; q < o.row_start[sr + 1]; ++q) {
          const float c2 = chi2_of(w, xyz[3 * (size_t)q + 1] - pr.y, xyz[3 * (size_t)q + 2] - pr.z);
          if (!(c2 <= cu.chi2_cut)) continue;
          if (g < 0 || c2 < best) { g = (int64_t)q; best = c2; }
        }
        is_new = g >= 0;
      }
      if (g >= 0) {
        if (!innovation(cu, pr, w, S00, S11) || !update(cu, pr, w, xyz[3 * (size_t)g + 1], xyz[3 * (size_t)g + 2], nx)) { if (k <= last) gained[ti] |= 0x80000000u; break; }
        st = nx; cur = k; miss = 0;
        if (is_new) { gained[ti] = (gained[ti] & 0x80000000u) | ((gained[ti] & 0x7fffffffu) + 1u); ++total; }
      } else if (k > last && ++miss > cu.max_row_gap) {
        break;
      }
    }
  }
  return total;
}

}  // extern "C"
