// kernels_merge.cu — NEXT-3: track sort, refit from the cluster lists and linking of track segments
// across sector boundaries ("the sector tracks are merged by the track merger", L98 "a
// fast sorting of the tracks in between of sector tracking and track merging", L102 "the track merger
// does a refit of the track"; G37-G40).  Runs after the output kernels on the track records
// and cluster-id lists in HBM; only cluster lists and row ranges enter (L102).  One lane per track
// (a few 10^4 per event, ~200 row steps each): the plain per-lane loops of the specification.
//   merge_rank  : G37 canonical order (sector, first_row, seed_cluster) by counting inside the sector:
//                 one warp per track over the sector's packed keys (written by merge_refit's prologue)
//   merge_refit : G38 outward and inward Kalman pass over the cluster list -> both end states; one lane
//                 per track (the two passes are a serial chain of ~2 x 90 row steps: 0.3 ms of latency)
//   merge_match : G39 chi2 of every admissible (segment, continuation) pair; one warp per segment scans
//                 the neighbouring sector's packed (ok, row_in) words 32 at a time, the few that pass the
//                 row test are evaluated; best continuation per segment in the warp, best origin per
//                 continuation by a 64-bit atomicMin
//   merge_link  : G40 a link is kept iff the two agree
//   merge_chain : G41 joint refit of every chain of linked segments, reported at its first segment
#include "kalman_math.cuh"

namespace tpcst {

// Packed per-track words for the scans: sort key (first_row << 32 | seed_cluster), (ok << 31 | row_in), and
// the first track of every sector (tracks are emitted in sector order; mg_sec[s] .. mg_sec[s + 1]).
__global__ void __launch_bounds__(128) merge_prepare(const __grid_constant__ Params p) {
  if (event_failed(p)) return;
  const uint32_t K = p.ctr->n_tracks, i = blockIdx.x * 128u + threadIdx.x;
  if (K == 0u) { if (i <= p.S) p.mg_sec[i] = 0u; return; }
  if (i >= K) return;
  const uint32_t sector = p.out_tracks[i].sector;
  p.mg_sortkey[i] = ((unsigned long long)p.out_tracks[i].first_row << 32) | p.out_tracks[i].seed_cluster;
  p.mg_best_a[i] = ~0ull;
  p.mg_best_b[i] = -1;
  const uint32_t prev = i ? p.out_tracks[i - 1u].sector + 1u : 0u;
  for (uint32_t s = prev; s <= sector; ++s) p.mg_sec[s] = i;          // sectors without tracks start here too
  if (i + 1u == K) for (uint32_t s = sector + 1u; s <= p.S; ++s) p.mg_sec[s] = K;
}

__global__ void __launch_bounds__(256) merge_rank(const __grid_constant__ Params p) {
  if (event_failed(p)) return;
  const uint32_t K = p.ctr->n_tracks, i = blockIdx.x * 8u + (threadIdx.x >> 5), lane = threadIdx.x & 31u;
  if (i >= K) return;
  const uint32_t sector = p.out_tracks[i].sector, lo = p.mg_sec[sector], hi = p.mg_sec[sector + 1u];
  const unsigned long long key = p.mg_sortkey[i];
  uint32_t r = 0;
  for (uint32_t j = lo + lane; j < hi; j += 32u) r += p.mg_sortkey[j] < key ? 1u : 0u;
  r = __reduce_add_sync(0xffffffffu, r);
  if (lane == 0u) p.mg_seg[i].rank = lo + r;
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
  if (event_failed(p)) return;
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
    // the next cluster (id, then y and z) is loaded while the current step is computed: the two dependent
    // round trips per cluster are off the serial chain of the fit
    uint32_t id_n = ids[1], id_nn = n > 2u ? ids[2] : 0u;
    float y_n = y1, z_n = z1;
    for (uint32_t j = 1; j < n && ok; ++j) {
      const uint32_t id = id_n;
      const float ym = y_n, zm = z_n;
      id_n = id_nn;
      if (j + 1u < n) { y_n = p.xyz[3 * (size_t)id_n + 1]; z_n = p.xyz[3 * (size_t)id_n + 2]; }
      if (j + 2u < n) id_nn = ids[j + 2u];
      const uint32_t k = row_of(p, srb, cur + 1u, id);
      float S00, S11, i00, i11;
      ok = kf_transport(p, st, p.tab[k].x - p.tab[cur].x, (float)(k - cur), pr) && kf_innov(p, pr, S00, S11, i00, i11) &&
           kf_update(p, pr, i00, i11, ym, zm, st);
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
    uint32_t id_d = ids[n - 2u], id_dd = n >= 3u ? ids[n - 3u] : 0u;
    float y_d = p.xyz[3 * (size_t)id_d + 1], z_d = p.xyz[3 * (size_t)id_d + 2];
    for (int32_t j = (int32_t)n - 2; j >= 0 && ok; --j) {
      const uint32_t id = id_d;
      const float ym = y_d, zm = z_d;
      id_d = id_dd;
      if (j >= 1) { y_d = p.xyz[3 * (size_t)id_d + 1]; z_d = p.xyz[3 * (size_t)id_d + 2]; }
      if (j >= 2) id_dd = ids[j - 2];
      uint32_t k = cur - 1u;
      while (id < p.row_start[srb + k]) --k;                   // row of the next id below
      float S00, S11, i00, i11;
      ok = kf_transport(p, st, p.tab[k].x - p.tab[cur].x, (float)(cur - k), pr) && kf_innov(p, pr, S00, S11, i00, i11);
      if (!ok) break;
      const float c2 = kf_chi2(i00, i11, ym - pr.y, zm - pr.z);
      ok = kf_update(p, pr, i00, i11, ym, zm, st);
      if (ok) { chi2 = chi2 + c2; cur = k; }
    }
  }
  sg->next = -1; sg->prev = -1; sg->ok = ok ? 1u : 0u; sg->match_chi2 = 0.0f;
  sg->row_in = ok ? row_in : 0u; sg->row_out = ok ? row_out : 0u;
  p.mg_word[i] = ok ? (0x80000000u | row_in) : 0u;
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

// G39 for one (segment, continuation) pair: chi2 or a negative value if the pair is not admissible.
__device__ __forceinline__ float match_chi2(const Params& p, const KState& rot, float xr, uint32_t last, uint32_t fr,
                                            const tpcst_merge_seg* sb) {
  KState pr;
  if (!kf_transport(p, rot, p.tab[fr].x - xr, (float)(fr - last), pr)) return -1.0f;
  // sum over the five parameters of d^2 / (C_ii(A') + C_ii(B)), left to right (plain IEEE division: the
  // variance of kappa is far below the range the short division sequence is checked for)
  const float d0 = pr.y - sb->in_par[0], d1 = pr.z - sb->in_par[1], d2 = pr.s - sb->in_par[2];
  const float d3 = pr.t - sb->in_par[3], d4 = pr.k - sb->in_par[4];
  const float v0 = pr.c00 + sb->in_cov[0], v1 = pr.c11 + sb->in_cov[2], v2 = pr.c22 + sb->in_cov[5];
  const float v3 = pr.c33 + sb->in_cov[9], v4 = pr.c44 + sb->in_cov[14];
  if (!(v0 > 0.0f) || !(v1 > 0.0f) || !(v2 > 0.0f) || !(v3 > 0.0f) || !(v4 > 0.0f)) return -1.0f;
  float chi2 = 0.0f;
  chi2 = chi2 + __fdiv_rn(d0 * d0, v0);
  chi2 = chi2 + __fdiv_rn(d1 * d1, v1);
  chi2 = chi2 + __fdiv_rn(d2 * d2, v2);
  chi2 = chi2 + __fdiv_rn(d3 * d3, v3);
  chi2 = chi2 + __fdiv_rn(d4 * d4, v4);
  return chi2 <= p.merge_chi2_cut ? chi2 : -1.0f;
}

__global__ void __launch_bounds__(256) merge_match(const __grid_constant__ Params p) {
  __shared__ uint32_t s_b[8][64];                          // per warp: candidates that passed the row test
  __shared__ uint8_t s_fr[8][64];
  if (event_failed(p)) return;
  const uint32_t K = p.ctr->n_tracks, wp = threadIdx.x >> 5, a = blockIdx.x * 8u + wp, lane = threadIdx.x & 31u;
  if (a >= K || (p.S % 18u) != 0u) return;
  const tpcst_merge_seg* const sa = p.mg_seg + a;
  if (!sa->ok) return;
  const uint32_t sector = p.out_tracks[a].sector, last = sa->row_out;
  KState out, rot;
  load_state(sa->out_par, sa->out_cov, out);
  const float sgn = out.y >= 0.0f ? 1.0f : -1.0f;
  const uint32_t half = sector / 18u, j = sector % 18u;
  const uint32_t nb = half * 18u + (sgn > 0.0f ? (j + 1u) % 18u : (j + 17u) % 18u);
  float xr;
  if (!gt_rotate(p, out, p.tab[last].x, sgn, rot, xr)) return;
  const uint32_t lo = p.mg_sec[nb], hi = p.mg_sec[nb + 1u];
  const uint32_t my_rank = sa->rank;
  unsigned long long best = ~0ull;                         // (chi2 bits << 32 | rank of the continuation): min = G40
  uint32_t best_b = 0u, cnt = 0u;
  // evaluates the first n <= 32 list entries, one per lane, and drops them from the list
  auto flush = [&](uint32_t n) {
    if (lane < n) {
      const uint32_t b = s_b[wp][lane];
      const tpcst_merge_seg* const sb = p.mg_seg + b;
      const float chi2 = match_chi2(p, rot, xr, last, s_fr[wp][lane], sb);
      if (chi2 >= 0.0f) {                                   // chi2 >= 0: its bits order like its value
        const unsigned long long hi32 = (unsigned long long)__float_as_uint(chi2) << 32;
        if ((hi32 | sb->rank) < best) { best = hi32 | sb->rank; best_b = b; }
        atomicMin(&p.mg_best_a[b], hi32 | my_rank);
      }
    }
    __syncwarp();
    uint32_t tb = 0u; uint8_t tf = 0u;
    const bool mv = lane + n < cnt;
    if (mv) { tb = s_b[wp][lane + n]; tf = s_fr[wp][lane + n]; }
    __syncwarp();
    if (mv) { s_b[wp][lane] = tb; s_fr[wp][lane] = tf; }
    __syncwarp();
    cnt -= n;
  };
  for (uint32_t b0 = lo; b0 < hi; b0 += 32u) {
    // 32 candidates per round: ok and 1 <= row_in(B) - row_out(A) <= merge_max_gap
    const uint32_t w = b0 + lane < hi ? p.mg_word[b0 + lane] : 0u;
    const uint32_t fr = w & 0xffu;
    const bool pass = (w >> 31) != 0u && fr > last && fr - last <= p.merge_max_gap;
    const uint32_t m = __ballot_sync(0xffffffffu, pass);
    if (pass) { const uint32_t pos = cnt + (uint32_t)__popc(m & ((1u << lane) - 1u)); s_b[wp][pos] = b0 + lane; s_fr[wp][pos] = (uint8_t)fr; }
    __syncwarp();
    cnt += (uint32_t)__popc(m);
    if (cnt >= 32u) flush(32u);
  }
  if (cnt) flush(cnt);
  // warp minimum of the lanes' best keys (total order: the rank is unique)
  unsigned long long wmin = best;
#pragma unroll
  for (int d = 16; d >= 1; d >>= 1) { const unsigned long long o = __shfl_xor_sync(0xffffffffu, wmin, d); wmin = o < wmin ? o : wmin; }
  if (wmin != ~0ull && best == wmin) { p.mg_best_b[a] = (int32_t)best_b; p.mg_chi_b[a] = __uint_as_float((uint32_t)(wmin >> 32)); }
}

__global__ void __launch_bounds__(128) merge_link(const __grid_constant__ Params p) {
  if (event_failed(p)) return;
  const uint32_t K = p.ctr->n_tracks, a = blockIdx.x * 128u + threadIdx.x;
  if (a >= K) return;
  const int32_t b = p.mg_best_b[a];
  if (b < 0) return;
  if ((uint32_t)p.mg_best_a[b] != p.mg_seg[a].rank) return;   // the best origin of b is somebody else
  p.mg_seg[a].next = b;
  p.mg_seg[a].match_chi2 = p.mg_chi_b[a];
  p.mg_seg[b].prev = (int32_t)a;
}

// G41: the merged track, reported at the first segment of every chain.  One lane per track; a chain of one
// segment repeats the segment's refit, a longer chain is refitted jointly over the cluster lists of its
// segments with the state rotated (G34) at the sector boundaries.  The outward pass over the first
// segment is that segment's own outward pass (same clusters, same arithmetic), so it starts from out_par.
__global__ void __launch_bounds__(128) merge_chain(const __grid_constant__ Params p) {
  if (event_failed(p)) return;
  const uint32_t K = p.ctr->n_tracks, h = blockIdx.x * 128u + threadIdx.x;
  if (h >= K) return;
  tpcst_merge_seg* const mh = p.mg_seg + h;
  uint32_t n_seg = 0u, n_cl = 0u;
  float chi2 = 0.0f;
  KState st;
  bool ok = mh->ok != 0u && mh->prev < 0;
  if (ok && mh->next < 0) {                                 // a chain of one segment
    n_seg = 1u; n_cl = p.out_tracks[h].n_clusters; chi2 = mh->chi2;
    load_state(mh->in_par, mh->in_cov, st);
  } else if (ok) {
    KState pr, rot;
    load_state(mh->out_par, mh->out_cov, st);
    uint32_t seg = h, prev_row = mh->row_out;
    float xcur = p.tab[prev_row].x;
    n_seg = 1u; n_cl = p.out_tracks[h].n_clusters;
    // ---- outward over the segments after the first
    for (int32_t nxt = mh->next; nxt >= 0 && ok; nxt = p.mg_seg[nxt].next) {
      const tpcst_track* const tk = p.out_tracks + nxt;
      const float sgn = ((tk->sector + 18u - p.out_tracks[seg].sector) % 18u) == 1u ? 1.0f : -1.0f;
      ok = gt_rotate(p, st, xcur, sgn, rot, xcur);
      if (!ok) break;
      st = rot;
      const uint32_t n = tk->n_clusters, srb = tk->sector * p.R;
      const uint32_t* const ids = p.out_ids + tk->first_cluster;
      uint32_t id_n = ids[0];                               // the next cluster is loaded while this one is fitted
      float y_n = p.xyz[3 * (size_t)id_n + 1], z_n = p.xyz[3 * (size_t)id_n + 2];
      for (uint32_t j = 0; j < n && ok; ++j) {
        const uint32_t id = id_n;
        const float ym = y_n, zm = z_n;
        if (j + 1u < n) { id_n = ids[j + 1u]; y_n = p.xyz[3 * (size_t)id_n + 1]; z_n = p.xyz[3 * (size_t)id_n + 2]; }
        const uint32_t k = j == 0u ? p.mg_seg[nxt].row_in : row_of(p, srb, prev_row + 1u, id);
        float S00, S11, i00, i11;
        ok = kf_transport(p, st, p.tab[k].x - xcur, (float)(k - prev_row), pr) && kf_innov(p, pr, S00, S11, i00, i11) &&
             kf_update(p, pr, i00, i11, ym, zm, st);
        xcur = p.tab[k].x; prev_row = k;
      }
      seg = (uint32_t)nxt; ++n_seg; n_cl += n;
    }
    // ---- inward from the top cluster of the last segment back to the first cluster of the head
    if (ok) {
      kf_reset_cov(p, st);
      const tpcst_track* const tk = p.out_tracks + seg;
      const uint32_t id = p.out_ids[tk->first_cluster + tk->n_clusters - 1u];
      const float ym = p.xyz[3 * (size_t)id + 1], zm = p.xyz[3 * (size_t)id + 2];
      float S00, S11, i00, i11;
      pr = st;
      ok = kf_innov(p, pr, S00, S11, i00, i11);
      if (ok) {
        chi2 = chi2 + kf_chi2(i00, i11, ym - pr.y, zm - pr.z);
        ok = kf_update(p, pr, i00, i11, ym, zm, st);
      }
    }
    bool top = true;
    for (int32_t sg = (int32_t)seg; sg >= 0 && ok; sg = p.mg_seg[sg].prev) {
      const tpcst_track* const tk = p.out_tracks + sg;
      const uint32_t n = tk->n_clusters, srb = tk->sector * p.R;
      const uint32_t* const ids = p.out_ids + tk->first_cluster;
      int32_t j = (int32_t)n - 1;
      if (top) { --j; top = false; }                        // the top cluster has been used
      else {                                                // back into this (lower) segment's frame
        const float sgn = ((p.out_tracks[seg].sector + 18u - tk->sector) % 18u) == 1u ? -1.0f : 1.0f;
        ok = gt_rotate(p, st, xcur, sgn, rot, xcur);
        if (!ok) break;
        st = rot;
      }
      uint32_t id_n = ids[j >= 0 ? j : 0];
      float y_n = p.xyz[3 * (size_t)id_n + 1], z_n = p.xyz[3 * (size_t)id_n + 2];
      for (; j >= 0 && ok; --j) {
        const uint32_t id = id_n;
        const float ym = y_n, zm = z_n;
        if (j >= 1) { id_n = ids[j - 1]; y_n = p.xyz[3 * (size_t)id_n + 1]; z_n = p.xyz[3 * (size_t)id_n + 2]; }
        uint32_t k;
        if (j == (int32_t)n - 1) k = p.mg_seg[sg].row_out;  // first cluster after the boundary
        else { k = prev_row - 1u; while (id < p.row_start[srb + k]) --k; }
        float S00, S11, i00, i11;
        ok = kf_transport(p, st, p.tab[k].x - xcur, (float)(prev_row - k), pr) && kf_innov(p, pr, S00, S11, i00, i11);
        if (!ok) break;
        const float c2 = kf_chi2(i00, i11, ym - pr.y, zm - pr.z);
        ok = kf_update(p, pr, i00, i11, ym, zm, st);
        if (ok) { chi2 = chi2 + c2; xcur = p.tab[k].x; prev_row = k; }
      }
      seg = (uint32_t)sg;
    }
  }
  if (ok) {
    mh->chain_n_seg = n_seg; mh->chain_n_clusters = n_cl; mh->chain_chi2 = chi2;
    store_state(st, mh->chain_par, mh->chain_cov);
  } else {
    mh->chain_n_seg = 0u; mh->chain_n_clusters = 0u; mh->chain_chi2 = 0.0f;
#pragma unroll
    for (int j = 0; j < 5; ++j) mh->chain_par[j] = 0.0f;
#pragma unroll
    for (int j = 0; j < 15; ++j) mh->chain_cov[j] = 0.0f;
  }
}

void launch_merge(const Params& p, cudaStream_t st, cudaEvent_t* ev) {
  const uint32_t nb = (p.kcap + 127u) / 128u, nw = (p.kcap + 7u) / 8u;     // lane per track / warp per track
  merge_prepare<<<nb, 128, 0, st>>>(p);
  merge_rank<<<nw, 256, 0, st>>>(p);    mark(ev, 16, st);
  merge_refit<<<nb, 128, 0, st>>>(p);   mark(ev, 17, st);
  merge_match<<<nw, 256, 0, st>>>(p);   mark(ev, 18, st);
  merge_link<<<nb, 128, 0, st>>>(p);    mark(ev, 19, st);
  merge_chain<<<nb, 128, 0, st>>>(p);   mark(ev, 20, st);
}

}  // namespace tpcst
