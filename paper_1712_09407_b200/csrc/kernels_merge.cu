// kernels_merge.cu — NEXT-3: track sort, refit from the cluster lists and linking of track segments
// across sector boundaries ("the sector tracks are merged by the track merger", L98 "a
// fast sorting of the tracks in between of sector tracking and track merging", L102 "the track merger
// does a refit of the track"; G37-G40).  Runs after the output kernels on the track records
// and cluster-id lists in HBM; only cluster lists and row ranges enter (L102).  One lane per track
// (a few 10^4 per event, ~200 row steps each): the plain per-lane loops of the specification.
//   merge_rank  : G37 canonical order (sector, first_row, seed_cluster) by counting inside the sector
//   merge_refit : G38 outward and inward Kalman pass over the cluster list -> both end states
//   merge_match : G39 chi2 of every admissible (segment, continuation) pair; the best continuation per
//                 segment stays in the lane, the best origin per continuation is a 64-bit atomicMin
//   merge_link  : G40 a link is kept iff the two agree
#include "kalman_math.cuh"

namespace tpcst {

// [lo, hi) of the tracks of `sector` in out_tracks (tracks are emitted in sector order).
__device__ __forceinline__ void sector_range(const Params& p, uint32_t K, uint32_t sector, uint32_t& lo, uint32_t& hi) {
  uint32_t a = 0, b = K;
  while (a < b) { const uint32_t m = (a + b) >> 1; if (p.out_tracks[m].sector < sector) a = m + 1; else b = m; }
  lo = a; b = K;
  while (a < b) { const uint32_t m = (a + b) >> 1; if (p.out_tracks[m].sector <= sector) a = m + 1; else b = m; }
  hi = a;
}

__global__ void __launch_bounds__(128) merge_rank(const __grid_constant__ Params p) {
  if (p.ctr->error) return;
  const uint32_t K = p.ctr->n_tracks, i = blockIdx.x * 128u + threadIdx.x;
  if (i >= K) return;
  const uint32_t sector = p.out_tracks[i].sector, fr = p.out_tracks[i].first_row, seed = p.out_tracks[i].seed_cluster;
  uint32_t lo, hi, r = 0;
  sector_range(p, K, sector, lo, hi);
  for (uint32_t j = lo; j < hi; ++j) {
    const uint32_t fj = p.out_tracks[j].first_row, sj = p.out_tracks[j].seed_cluster;
    r += (fj < fr || (fj == fr && sj < seed)) ? 1u : 0u;
  }
  p.mg_seg[i].rank = lo + r;
  p.mg_best_a[i] = ~0ull;
  p.mg_best_b[i] = -1;
}

__device__ __forceinline__ void store_state(const KState& a, float* par, float* cov) {
  par[0] = a.y; par[1] = a.z; par[2] = a.s; par[3] = a.t; par[4] = a.k;
#pragma unroll
  for (int i = 0; i < 15; ++i) cov[i] = 0.0f;
  cov[0] = a.c00; cov[2] = a.c11; cov[3] = a.c20; cov[5] = a.c22; cov[7] = a.c31; cov[9] = a.c33;
  cov[10] = a.c40; cov[12] = a.c42; cov[14] = a.c44;
}
__device__ __forceinline__ void load_state(const float* par, const float* cov, KState& a) {
  a.y = par[0]; a.z = par[1]; a.s = par[2]; a.t = par[3]; a.k = par[4];
  a.c00 = cov[0]; a.c11 = cov[2]; a.c20 = cov[3]; a.c22 = cov[5]; a.c31 = cov[7]; a.c33 = cov[9];
  a.c40 = cov[10]; a.c42 = cov[12]; a.c44 = cov[14];
}

// Walks a cluster-id list (ascending rows): row of the next id, starting the search at row k.
__device__ __forceinline__ uint32_t row_of(const Params& p, uint32_t srb, uint32_t k, uint32_t id) {
  while (id >= p.row_start[srb + k + 1u]) ++k;
  return k;
}

__global__ void __launch_bounds__(128) merge_refit(const __grid_constant__ Params p) {
  if (p.ctr->error) return;
  const uint32_t K = p.ctr->n_tracks, i = blockIdx.x * 128u + threadIdx.x;
  if (i >= K) return;
  tpcst_merge_seg* const sg = p.mg_seg + i;
  const tpcst_track* const tk = p.out_tracks + i;
  const uint32_t n = tk->n_clusters, srb = tk->sector * p.R;
  const uint32_t* const ids = p.out_ids + tk->first_cluster;
  bool ok = n >= 2u;
  KState st, pr, top;
  float chi2 = 0.0f;
  uint32_t row_in = 0u, row_out = 0u;
  if (ok) {
    // G38 outward pass: state from the first two clusters (G15), then cluster by cluster
    uint32_t cur = row_of(p, srb, tk->first_row, ids[0]);   // the cluster on first_row may have gone to another track
    row_in = cur;
    const uint32_t k1 = row_of(p, srb, cur + 1u, ids[1]);
    const float y0 = p.xyz[3 * (size_t)ids[0] + 1], z0 = p.xyz[3 * (size_t)ids[0] + 2];
    const float y1 = p.xyz[3 * (size_t)ids[1] + 1], z1 = p.xyz[3 * (size_t)ids[1] + 2];
    const float dx = p.tab[k1].x - p.tab[cur].x;
    const float m = (y1 - y0) / dx;
    const float q2 = sqrtf(1.0f + m * m);
    st.y = y0; st.z = z0; st.s = m / q2; st.t = (z1 - z0) / (dx * q2); st.k = 0.0f;
    kf_reset_cov(p, st);
    for (uint32_t j = 1; j < n && ok; ++j) {
      const uint32_t id = ids[j], k = row_of(p, srb, cur + 1u, id);
      float S00, S11, i00, i11;
      ok = kf_transport(p, st, p.tab[k].x - p.tab[cur].x, (float)(k - cur), pr) && kf_innov(p, pr, S00, S11, i00, i11) &&
           kf_update(p, pr, i00, i11, p.xyz[3 * (size_t)id + 1], p.xyz[3 * (size_t)id + 2], st);
      cur = k;
    }
    top = st;
    row_out = cur;
    // inward pass (G22.2): covariance reset, update with the top cluster, then down the list
    if (ok) {
      kf_reset_cov(p, st);
      float S00, S11, i00, i11;
      const uint32_t id = ids[n - 1u];
      const float ym = p.xyz[3 * (size_t)id + 1], zm = p.xyz[3 * (size_t)id + 2];
      pr = st;
      ok = kf_innov(p, pr, S00, S11, i00, i11);
      if (ok) {
        chi2 = chi2 + kf_chi2(i00, i11, ym - pr.y, zm - pr.z);
        ok = kf_update(p, pr, i00, i11, ym, zm, st);
      }
    }
    for (int32_t j = (int32_t)n - 2; j >= 0 && ok; --j) {
      const uint32_t id = ids[j];
      uint32_t k = cur - 1u;
      while (id < p.row_start[srb + k]) --k;                   // row of the next id below
      float S00, S11, i00, i11;
      ok = kf_transport(p, st, p.tab[k].x - p.tab[cur].x, (float)(cur - k), pr) && kf_innov(p, pr, S00, S11, i00, i11);
      if (!ok) break;
      const float ym = p.xyz[3 * (size_t)id + 1], zm = p.xyz[3 * (size_t)id + 2];
      const float c2 = kf_chi2(i00, i11, ym - pr.y, zm - pr.z);
      ok = kf_update(p, pr, i00, i11, ym, zm, st);
      if (ok) { chi2 = chi2 + c2; cur = k; }
    }
  }
  sg->next = -1; sg->prev = -1; sg->ok = ok ? 1u : 0u; sg->match_chi2 = 0.0f;
  sg->row_in = ok ? row_in : 0u; sg->row_out = ok ? row_out : 0u;
  if (ok) {
    sg->chi2 = chi2;
    store_state(st, sg->in_par, sg->in_cov);
    store_state(top, sg->out_par, sg->out_cov);
  } else {
    sg->chi2 = 0.0f;
#pragma unroll
    for (int j = 0; j < 5; ++j) { sg->in_par[j] = 0.0f; sg->out_par[j] = 0.0f; }
#pragma unroll
    for (int j = 0; j < 15; ++j) { sg->in_cov[j] = 0.0f; sg->out_cov[j] = 0.0f; }
  }
}

__global__ void __launch_bounds__(128) merge_match(const __grid_constant__ Params p) {
  if (p.ctr->error) return;
  const uint32_t K = p.ctr->n_tracks, a = blockIdx.x * 128u + threadIdx.x;
  if (a >= K || (p.S % 18u) != 0u) return;
  const tpcst_merge_seg* const sa = p.mg_seg + a;
  if (!sa->ok) return;
  const uint32_t sector = p.out_tracks[a].sector, last = sa->row_out;
  KState out, rot, pr;
  load_state(sa->out_par, sa->out_cov, out);
  const float sgn = out.y >= 0.0f ? 1.0f : -1.0f;
  const uint32_t half = sector / 18u, j = sector % 18u;
  const uint32_t nb = half * 18u + (sgn > 0.0f ? (j + 1u) % 18u : (j + 17u) % 18u);
  float xr;
  if (!gt_rotate(p, out, p.tab[last].x, sgn, rot, xr)) return;
  uint32_t lo, hi;
  sector_range(p, K, nb, lo, hi);
  const uint32_t my_rank = sa->rank;
  int32_t best = -1;
  uint32_t best_rank = 0u;
  float best_chi2 = 0.0f;
  for (uint32_t b = lo; b < hi; ++b) {
    const tpcst_merge_seg* const sb = p.mg_seg + b;
    const uint32_t fr = sb->row_in;
    if (!sb->ok || !(fr > last && fr - last <= p.merge_max_gap)) continue;
    if (!kf_transport(p, rot, p.tab[fr].x - xr, (float)(fr - last), pr)) continue;
    // G39: sum over the five parameters of d^2 / (C_ii(A') + C_ii(B)), left to right (plain IEEE division:
    // the variance of kappa is far below the range the short division sequence is checked for)
    const float d0 = pr.y - sb->in_par[0], d1 = pr.z - sb->in_par[1], d2 = pr.s - sb->in_par[2];
    const float d3 = pr.t - sb->in_par[3], d4 = pr.k - sb->in_par[4];
    const float v0 = pr.c00 + sb->in_cov[0], v1 = pr.c11 + sb->in_cov[2], v2 = pr.c22 + sb->in_cov[5];
    const float v3 = pr.c33 + sb->in_cov[9], v4 = pr.c44 + sb->in_cov[14];
    if (!(v0 > 0.0f) || !(v1 > 0.0f) || !(v2 > 0.0f) || !(v3 > 0.0f) || !(v4 > 0.0f)) continue;
    float chi2 = 0.0f;
    chi2 = chi2 + __fdiv_rn(d0 * d0, v0);
    chi2 = chi2 + __fdiv_rn(d1 * d1, v1);
    chi2 = chi2 + __fdiv_rn(d2 * d2, v2);
    chi2 = chi2 + __fdiv_rn(d3 * d3, v3);
    chi2 = chi2 + __fdiv_rn(d4 * d4, v4);
    if (!(chi2 <= p.merge_chi2_cut)) continue;
    const uint32_t rb = sb->rank;
    if (best < 0 || chi2 < best_chi2 || (chi2 == best_chi2 && rb < best_rank)) { best = (int32_t)b; best_chi2 = chi2; best_rank = rb; }
    atomicMin(&p.mg_best_a[b], ((unsigned long long)__float_as_uint(chi2) << 32) | my_rank);   // chi2 >= 0: bits order like values
  }
  p.mg_best_b[a] = best;
  p.mg_chi_b[a] = best_chi2;
}

__global__ void __launch_bounds__(128) merge_link(const __grid_constant__ Params p) {
  if (p.ctr->error) return;
  const uint32_t K = p.ctr->n_tracks, a = blockIdx.x * 128u + threadIdx.x;
  if (a >= K) return;
  const int32_t b = p.mg_best_b[a];
  if (b < 0) return;
  if ((uint32_t)p.mg_best_a[b] != p.mg_seg[a].rank) return;   // the best origin of b is somebody else
  p.mg_seg[a].next = b;
  p.mg_seg[a].match_chi2 = p.mg_chi_b[a];
  p.mg_seg[b].prev = (int32_t)a;
}

void launch_merge(const Params& p, cudaStream_t st, cudaEvent_t* ev) {
  const uint32_t nb = (p.kcap + 127u) / 128u;
  merge_rank<<<nb, 128, 0, st>>>(p);    mark(ev, 16, st);
  merge_refit<<<nb, 128, 0, st>>>(p);   mark(ev, 17, st);
  merge_match<<<nb, 128, 0, st>>>(p);   mark(ev, 18, st);
  merge_link<<<nb, 128, 0, st>>>(p);    mark(ev, 19, st);
}

}  // namespace tpcst
