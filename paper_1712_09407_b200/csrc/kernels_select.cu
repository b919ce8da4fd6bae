// kernels_select.cu — a6 tracklet selection (G26) and a7 track
// output (L52, L102; G27/G28).
//   select_claim   : every tracklet with nhits >= min_clusters claims its hits with a 64-bit
//                    atomicMax on a packed key -> deterministic owner per cluster (removes the
//                    nondeterminism the paper describes in L78)
//   select_collect : per tracklet, count owned hits, apply the cuts, per-block sums
//   scan_partials  : exclusive scan of the block sums -> output offsets
//   write_tracks   : ordered compaction: track records + contiguous cluster-id lists
#include "tpcst_internal.h"

namespace tpcst {

__device__ __forceinline__ uint32_t float_order_bits(float w) {   // order-preserving float -> uint32
  const uint32_t b = __float_as_uint(w);
  return (b & 0x80000000u) ? ~b : (b | 0x80000000u);
}

// Claim key of tracklet t (rank t_local inside its sector).  Mode 0: (nhits << 24 | ~t_local) —
// longest wins, first wins on ties (L46, L78).  Mode 1: weight n*(alpha - chi2/ndf) (L88), then
// lower id.  The high word orders, the low word stores what `owner` reports to the caller.
__device__ __forceinline__ unsigned long long claim_key(const Params& p, uint32_t nh, float chi2, uint32_t t_local) {
  if (p.select_mode == 0u) {
    const uint32_t k = (nh << 24) | (0xFFFFFFu - t_local);
    return ((unsigned long long)k << 32) | k;
  }
  const float n = (float)nh;
  const float ndf = 2.0f * n - 5.0f;
  const float w = n * (p.alpha - chi2 / ndf);
  return ((unsigned long long)float_order_bits(w) << 32) | (unsigned long long)(0xFFFFFFFFu - t_local);
}
// What the tests see as the owner value: mode 0 the packed key, mode 1 t_local + 1.
__device__ __forceinline__ uint32_t owner_value(const Params& p, unsigned long long key) {
  if (key == 0ull) return 0u;
  return p.select_mode == 0u ? (uint32_t)key : (0xFFFFFFFFu - (uint32_t)key) + 1u;
}

// Fields of t_rows[t] (written by construct_tracklets).
__device__ __forceinline__ uint32_t tr_first(uint32_t r) { return r & 0xffu; }
__device__ __forceinline__ uint32_t tr_last(uint32_t r) { return (r >> 8) & 0xffu; }
__device__ __forceinline__ uint32_t tr_nhits(uint32_t r) { return (r >> 16) & 0xffu; }
__device__ __forceinline__ uint32_t tr_sector(uint32_t r) { return r >> 24; }

// The selection kernels work on ITEMS = (tracklet, group of 32 rows): one warp iteration takes a
// chunk of 32 consecutive items; lane j fetches the header t_rows of item j (coalesced), a ballot
// picks the items of tracklets long enough to claim (G26) whose group overlaps [first_row,
// last_row], and the warp walks those, lane = row inside the group: one coalesced 64-byte read of
// hits[t][32g ..], the slab start of each row, then owner[] there.  Nothing waits on the walk of
// another item, so the gathers of many items are in flight at once (the first version walked the
// tracklets of a warp one after the other and was latency-bound: 15 % issue utilisation, ncu r01d).
struct ItemHdr { uint32_t rows, t; unsigned long long key; };

__device__ __forceinline__ uint32_t item_chunk(const Params& p, uint32_t chunk, uint32_t lane, uint32_t T, uint32_t& my_t,
                                               uint32_t& my_g, uint32_t& my_rows) {
  const uint32_t item = chunk * 32u + lane;
  my_t = item / p.hit_groups;
  my_g = item - my_t * p.hit_groups;
  my_rows = my_t < T ? p.t_rows[my_t] : 0u;
  bool walk = tr_nhits(my_rows) >= p.min_clusters && my_g * 32u <= tr_last(my_rows) && my_g * 32u + 31u >= tr_first(my_rows);
  if (p.sel_round != 0u && walk) walk = (p.t_kept[my_t] >> 31) != 0u;      // G26b: the second round is among the accepted
  return __ballot_sync(0xffffffffu, walk);
}

template <bool kCount>
__global__ void __launch_bounds__(256) select_claim(const __grid_constant__ Params p) {
  if (event_failed(p)) return;
  const uint32_t T = p.ctr->n_tracklets, lane = threadIdx.x & 31u;
  const uint32_t n_chunks = (T * p.hit_groups + 31u) / 32u, n_warps = gridDim.x * (blockDim.x >> 5);
  uint32_t n_claimed = 0;
  for (uint32_t chunk = blockIdx.x * (blockDim.x >> 5) + (threadIdx.x >> 5); chunk < n_chunks; chunk += n_warps) {
    uint32_t my_t, my_g, my_rows;
    uint32_t todo = item_chunk(p, chunk, lane, T, my_t, my_g, my_rows);
    unsigned long long my_key = 0ull;
    if ((todo >> lane) & 1u) my_key = claim_key(p, tr_nhits(my_rows), p.t_chi2[my_t], my_t - p.row_off[tr_sector(my_rows) * p.R]);
    // four items at a time: their hit rows are fetched together (independent 64-byte loads), then claimed; a warp
    // that takes one item per round trip spends its time waiting for that one load
    while (todo) {
      uint32_t h[4], pos[4];
      unsigned long long key[4];
#pragma unroll
      for (int u = 0; u < 4; ++u) {
        h[u] = 0xffffu; pos[u] = 0u; key[u] = 0ull;
        if (todo) {
          const int j = __ffs(todo) - 1;
          todo &= todo - 1u;
          const uint32_t rows = __shfl_sync(0xffffffffu, my_rows, j), t = __shfl_sync(0xffffffffu, my_t, j);
          const uint32_t k = __shfl_sync(0xffffffffu, my_g, j) * 32u + lane;
          key[u] = __shfl_sync(0xffffffffu, my_key, j);
          if (k >= tr_first(rows) && k <= tr_last(rows)) {
            h[u] = p.hits[(size_t)t * p.hit_stride + k];
            const uint32_t sr = tr_sector(rows) * p.R + k;
            pos[u] = pstart(p.row_start[sr], sr);
          }
        }
      }
#pragma unroll
      for (int u = 0; u < 4; ++u) {
        if (h[u] == 0xffffu) continue;
        owner_claim(p, pos[u] + h[u], key[u]);
        if (kCount) ++n_claimed;
      }
    }
  }
  if (kCount) { __syncwarp(); count_add_warp(&p.ctr->claimed_hits, n_claimed); }
}

// Kept hits of every item = hits whose owner is the tracklet's own key -> t_grp[t][g] (one byte per
// group of every claiming tracklet; 0 for a group outside its row range).
__global__ void __launch_bounds__(256) select_collect(const __grid_constant__ Params p) {
  if (event_failed(p)) return;
  const uint32_t T = p.ctr->n_tracklets, lane = threadIdx.x & 31u;
  const uint32_t n_chunks = (T * p.hit_groups + 31u) / 32u, n_warps = gridDim.x * (blockDim.x >> 5);
  for (uint32_t chunk = blockIdx.x * (blockDim.x >> 5) + (threadIdx.x >> 5); chunk < n_chunks; chunk += n_warps) {
    uint32_t my_t, my_g, my_rows;
    uint32_t todo = item_chunk(p, chunk, lane, T, my_t, my_g, my_rows);
    unsigned long long my_key = 0ull;
    if ((todo >> lane) & 1u) my_key = claim_key(p, tr_nhits(my_rows), p.t_chi2[my_t], my_t - p.row_off[tr_sector(my_rows) * p.R]);
    uint32_t my_kept = 0, my_mask = 0;
    const bool claims = my_t < T && tr_nhits(my_rows) >= p.min_clusters && (p.sel_round == 0u || (p.t_kept[my_t] >> 31) != 0u);
    for (; todo; todo &= todo - 1u) {
      const int j = __ffs(todo) - 1;
      const uint32_t rows = __shfl_sync(0xffffffffu, my_rows, j), t = __shfl_sync(0xffffffffu, my_t, j);
      const uint32_t k = __shfl_sync(0xffffffffu, my_g, j) * 32u + lane;
      const unsigned long long key = __shfl_sync(0xffffffffu, my_key, j);
      bool kept = false;
      if (k >= tr_first(rows) && k <= tr_last(rows)) {
        const uint32_t h = p.hits[(size_t)t * p.hit_stride + k];
        if (h != 0xffffu) {
          const uint32_t sr = tr_sector(rows) * p.R + k;
          kept = owner_get(p, pstart(p.row_start[sr], sr) + h) == key;
        }
      }
      const uint32_t m = __ballot_sync(0xffffffffu, kept);
      if ((int)lane == j) { my_kept = (uint32_t)__popc(m); my_mask = m; }
    }
    if (claims) {
      p.t_grp[(size_t)my_t * 8u + my_g] = (uint8_t)my_kept;
      p.t_mask[(size_t)my_t * 8u + my_g] = my_mask;          // which rows of the group: write_ids does not ask owner[] again
    }
  }
}

// Per tracklet: kept = sum over its groups; cuts (kept >= min_clusters, |q/pT| <= 1/min_pt); per-CTA sums.
__global__ void __launch_bounds__(kKalmanBlock) select_accept(const __grid_constant__ Params p) {
  __shared__ uint32_t s_acc[kKalmanBlock / 32], s_kept[kKalmanBlock / 32];
  if (event_failed(p)) return;
  const uint32_t T = p.ctr->n_tracklets;
  if (blockIdx.x * kKalmanBlock >= T) return;
  const uint32_t t = blockIdx.x * kKalmanBlock + threadIdx.x, lane = threadIdx.x & 31u, w = threadIdx.x >> 5;
  uint32_t kept = 0, acc = 0;
  if (t < T && tr_nhits(p.t_rows[t]) >= p.min_clusters && (p.sel_round == 0u || (p.t_kept[t] >> 31) != 0u)) {
    const unsigned long long g8 = *reinterpret_cast<const unsigned long long*>(p.t_grp + (size_t)t * 8u);
    for (uint32_t g = 0; g < p.hit_groups; ++g) kept += (uint32_t)(g8 >> (8u * g)) & 0xffu;
    const float qpt = (0.0f - p.t_par[4 * (size_t)p.tcap + t]) / p.kbz;   // G14
    acc = (kept >= p.min_clusters && fabsf(qpt) <= p.max_qpt) ? 1u : 0u;
  }
  if (t < T) p.t_kept[t] = kept | (acc << 31);
  const uint32_t sum_acc = __reduce_add_sync(0xffffffffu, acc);
  const uint32_t sum_kept = __reduce_add_sync(0xffffffffu, acc ? kept : 0u);
  if (lane == 0) { s_acc[w] = sum_acc; s_kept[w] = sum_kept; }
  __syncthreads();
  if (threadIdx.x == 0) {
    uint32_t ta = 0, tk = 0;
    for (int i = 0; i < kKalmanBlock / 32; ++i) { ta += s_acc[i]; tk += s_kept[i]; }
    const uint32_t nblk = (p.tcap + kKalmanBlock - 1) / kKalmanBlock;
    p.partials[blockIdx.x] = ta;
    p.partials[nblk + blockIdx.x] = tk;
  }
}

// Exclusive scan (in place) of the per-block sums of the blocks that hold tracklets.
__global__ void __launch_bounds__(1024) scan_partials(const __grid_constant__ Params p) {
  __shared__ uint32_t wa[32], wk[32];
  if (event_failed(p)) return;
  const uint32_t T = p.ctr->n_tracklets;
  const uint32_t nblk = (p.tcap + kKalmanBlock - 1) / kKalmanBlock;
  const uint32_t used = (T + kKalmanBlock - 1) / kKalmanBlock;
  const int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
  // every thread owns a contiguous chunk of the per-CTA sums; the chunk sums are scanned across the block
  const uint32_t chunk = (used + 1023u) / 1024u, i0 = min(threadIdx.x * chunk, used), i1 = min(i0 + chunk, used);
  uint32_t sa = 0, sk = 0;
  for (uint32_t i = i0; i < i1; ++i) { sa += p.partials[i]; sk += p.partials[nblk + i]; }
  uint32_t ia = sa, ik = sk;
#pragma unroll
  for (int d = 1; d < 32; d <<= 1) {
    const uint32_t oa = __shfl_up_sync(0xffffffffu, ia, d), ok = __shfl_up_sync(0xffffffffu, ik, d);
    if (lane >= d) { ia += oa; ik += ok; }
  }
  if (lane == 31) { wa[w] = ia; wk[w] = ik; }
  __syncthreads();
  uint32_t ba = 0, bk = 0, ta = 0, tk = 0;
  for (int j = 0; j < 32; ++j) { if (j < w) { ba += wa[j]; bk += wk[j]; } ta += wa[j]; tk += wk[j]; }
  uint32_t ra = ba + ia - sa, rk = bk + ik - sk;
  for (uint32_t i = i0; i < i1; ++i) {
    const uint32_t va = p.partials[i], vk = p.partials[nblk + i];
    p.partials[i] = ra; p.partials[nblk + i] = rk;
    ra += va; rk += vk;
  }
  if (threadIdx.x == 0) {
    if (ta > p.kcap || tk > p.max_clusters) { atomicOr(&p.ctr->error, kErrTrackCap); ta = 0; tk = 0; }
    p.ctr->n_tracks = ta;
    p.ctr->n_ids = tk;
  }
}

// Ordered compaction, part 1.  One thread per tracklet: block-local exclusive scan of (accepted,
// kept) on top of the scanned per-CTA sums -> track index and first cluster-id slot; the accepted
// threads write their track record and t_ci[t] (0xffffffff = not accepted).
__global__ void __launch_bounds__(kKalmanBlock) write_tracks(const __grid_constant__ Params p) {
  __shared__ uint32_t s_a[kKalmanBlock / 32], s_k[kKalmanBlock / 32];
  if (event_failed(p)) return;
  const uint32_t t = blockIdx.x * kKalmanBlock + threadIdx.x;
  const uint32_t T = p.ctr->n_tracklets;
  if (blockIdx.x * kKalmanBlock >= T) return;
  const uint32_t kw = t < T ? p.t_kept[t] : 0u;
  const uint32_t acc = kw >> 31, kept = acc ? (kw & 0x7fffffffu) : 0u;
  const int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
  uint32_t ia = acc, ik = kept;
#pragma unroll
  for (int d = 1; d < 32; d <<= 1) {
    const uint32_t oa = __shfl_up_sync(0xffffffffu, ia, d), ok = __shfl_up_sync(0xffffffffu, ik, d);
    if (lane >= d) { ia += oa; ik += ok; }
  }
  if (lane == 31) { s_a[w] = ia; s_k[w] = ik; }
  __syncthreads();
  uint32_t ba = 0, bk = 0;
  for (int j = 0; j < w; ++j) { ba += s_a[j]; bk += s_k[j]; }
  const uint32_t nblk = (p.tcap + kKalmanBlock - 1) / kKalmanBlock;
  const size_t hs = p.tcap;
  uint32_t ci = 0xffffffffu;
  if (acc) {
    const uint32_t ti = p.partials[blockIdx.x] + ba + ia - 1u;           // track index
    ci = p.partials[nblk + blockIdx.x] + bk + ik - kept;                 // first cluster id slot
    const uint32_t rows = p.t_rows[t];
    tpcst_track tk;
    tk.sector = tr_sector(rows); tk.first_row = tr_first(rows); tk.last_row = tr_last(rows);
    tk.n_clusters = kept; tk.first_cluster = ci;
    tk.seed_cluster = p.s_orig[p.t_seed[t]];
    tk.x_ref = p.tab[p.max_passes > 2u ? p.t_ref[t] : tk.first_row].x;   // G22d: where the last kept pass ended
    tk.y = p.t_par[t]; tk.z = p.t_par[hs + t]; tk.sinphi = p.t_par[2 * hs + t]; tk.dzds = p.t_par[3 * hs + t];
    tk.qpt = (0.0f - p.t_par[4 * hs + t]) / p.kbz;
#pragma unroll
    for (int i = 0; i < 15; ++i) tk.cov[i] = 0.0f;
    tk.cov[0] = p.t_cov[t]; tk.cov[3] = p.t_cov[hs + t]; tk.cov[5] = p.t_cov[2 * hs + t];
    tk.cov[10] = p.t_cov[3 * hs + t]; tk.cov[12] = p.t_cov[4 * hs + t]; tk.cov[14] = p.t_cov[5 * hs + t];
    tk.cov[2] = p.t_cov[6 * hs + t]; tk.cov[7] = p.t_cov[7 * hs + t]; tk.cov[9] = p.t_cov[8 * hs + t];
    tk.chi2 = p.t_chi2[t];
    p.out_tracks[ti] = tk;
    if (p.global_tracking) p.trk_t[ti] = t;
  }
  if (t < T) p.t_ci[t] = ci;
}

// Ordered compaction, part 2: the kept clusters of every accepted tracklet in ascending row order ->
// its contiguous cluster-id list.  Items as above; an item's first slot is the track's first slot
// plus the kept counts of the lower groups (t_grp); the kept rows of the group are the mask select_collect left.
__global__ void __launch_bounds__(256) write_ids(const __grid_constant__ Params p) {
  if (event_failed(p)) return;
  const uint32_t T = p.ctr->n_tracklets, lane = threadIdx.x & 31u;
  const uint32_t n_chunks = (T * p.hit_groups + 31u) / 32u, n_warps = gridDim.x * (blockDim.x >> 5);
  for (uint32_t chunk = blockIdx.x * (blockDim.x >> 5) + (threadIdx.x >> 5); chunk < n_chunks; chunk += n_warps) {
    uint32_t my_t, my_g, my_rows;
    uint32_t todo = item_chunk(p, chunk, lane, T, my_t, my_g, my_rows);
    uint32_t my_slot = 0xffffffffu, my_mask = 0u;
    if ((todo >> lane) & 1u) {
      my_slot = p.t_ci[my_t];
      if (my_slot != 0xffffffffu) {
        my_mask = p.t_mask[(size_t)my_t * 8u + my_g];
        const unsigned long long g8 = *reinterpret_cast<const unsigned long long*>(p.t_grp + (size_t)my_t * 8u);
        for (uint32_t g = 0; g < my_g; ++g) my_slot += (uint32_t)(g8 >> (8u * g)) & 0xffu;
      }
    }
    todo = __ballot_sync(0xffffffffu, my_slot != 0xffffffffu);
    while (todo) {                                                      // four items at a time (see select_claim)
      uint32_t h[4], pos[4], dst[4];
#pragma unroll
      for (int u = 0; u < 4; ++u) {
        h[u] = 0xffffu; pos[u] = 0u; dst[u] = 0u;
        if (todo) {
          const int j = __ffs(todo) - 1;
          todo &= todo - 1u;
          const uint32_t rows = __shfl_sync(0xffffffffu, my_rows, j), t = __shfl_sync(0xffffffffu, my_t, j);
          const uint32_t k = __shfl_sync(0xffffffffu, my_g, j) * 32u + lane;
          const uint32_t c0 = __shfl_sync(0xffffffffu, my_slot, j);
          const uint32_t m = __shfl_sync(0xffffffffu, my_mask, j);       // kept rows of the group (select_collect)
          if ((m >> lane) & 1u) {
            h[u] = p.hits[(size_t)t * p.hit_stride + k];
            const uint32_t sr = tr_sector(rows) * p.R + k;
            pos[u] = pstart(p.row_start[sr], sr);
            dst[u] = c0 + (uint32_t)__popc(m & ((1u << lane) - 1u));
          }
        }
      }
      uint32_t o[4];
#pragma unroll
      for (int u = 0; u < 4; ++u) o[u] = h[u] != 0xffffu ? p.s_orig[pos[u] + h[u]] : 0u;
#pragma unroll
      for (int u = 0; u < 4; ++u) if (h[u] != 0xffffu) p.out_ids[dst[u]] = o[u];
    }
  }
}

// Used by the debug path: owner value per ORIGINAL cluster index.
__global__ void owners_to_orig(const __grid_constant__ Params p, uint32_t* out) {
  const uint32_t sr = blockIdx.x;
  const uint32_t g0 = p.row_start[sr], n = p.row_start[sr + 1] - g0;
  const uint32_t p0 = pstart(g0, sr);
  for (uint32_t i = threadIdx.x; i < n; i += blockDim.x) out[p.s_orig[p0 + i]] = owner_value(p, owner_get(p, p0 + i));
}
void launch_owners_to_orig(const Params& p, uint32_t* out, cudaStream_t st) {
  owners_to_orig<<<p.S * p.R, 128, 0, st>>>(p, out);
}

__global__ void __launch_bounds__(256) clear_owner(const __grid_constant__ Params p) {
  ulonglong2* const o = reinterpret_cast<ulonglong2*>(p.owner);
  for (uint32_t i = blockIdx.x * 256u + threadIdx.x; i < p.npad / 2u; i += gridDim.x * 256u) o[i] = make_ulonglong2(0ull, 0ull);
}

void launch_select(const Params& p, cudaStream_t st, cudaEvent_t* ev, bool count) {
  const uint32_t nb = (p.tcap + kKalmanBlock - 1) / kKalmanBlock;
  if (count) select_claim<true><<<p.sel_grid, 256, 0, st>>>(p);
  else select_claim<false><<<p.sel_grid, 256, 0, st>>>(p);
  mark(ev, 7, st);
  select_collect<<<p.sel_grid, 256, 0, st>>>(p);             mark(ev, 8, st);
  select_accept<<<nb, kKalmanBlock, 0, st>>>(p);             mark(ev, 9, st);
  if (p.select_rounds >= 2u) {
    // G26b: owners cleared, then the same three kernels among the accepted tracklets (their times
    // are added to the per-kernel events of the first round's successor, scan_partials)
    Params q = p;
    q.sel_round = 1u;
    clear_owner<<<p.sel_grid, 256, 0, st>>>(p);           // a kernel, not cudaMemsetAsync: the copy engines are busy with the next event's input
    select_claim<false><<<p.sel_grid, 256, 0, st>>>(q);
    select_collect<<<p.sel_grid, 256, 0, st>>>(q);
    select_accept<<<nb, kKalmanBlock, 0, st>>>(q);
  }
  scan_partials<<<1, 1024, 0, st>>>(p);                      mark(ev, 10, st);
  write_tracks<<<nb, kKalmanBlock, 0, st>>>(p);              mark(ev, 11, st);
  write_ids<<<p.sel_grid, 256, 0, st>>>(p);                  mark(ev, 12, st);
}

}  // namespace tpcst
