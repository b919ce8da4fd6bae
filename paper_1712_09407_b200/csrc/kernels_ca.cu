// kernels_ca.cu — the cellular-automaton half of the sector tracker on sm_100a:
//   bin_rows        (a1, "initialization"; G4/G5)
//   find_neighbours (a2, L40; G6-G10)
//   evolve_links    (a3, L41; G11)
//   find_starts     (a4, L43; G12)  + scan_rows (tracklet ids by ordered compaction)
// One CTA per (sector,row) for every kernel: a row slab (~5 KB of float2 + a ~6 KB bin table) is
// the natural tile, 36*159 = 5724 CTAs = 38.7 per SM.  All arithmetic that decides an integer is
// fp32 with one rounding per operation (compiled with -fmad=false), in the order DESIGN.md fixes.
#include "tpcst_internal.h"

namespace tpcst {

// G4: f = (v + off) * inv; clamp; truncate.  NaN -> 0.
__device__ __forceinline__ uint32_t bin_coord(float v, float off, float inv, uint32_t n) {
  const float f = (v + off) * inv;
  if (!(f >= 0.0f)) return 0u;
  if (f >= (float)(n - 1u)) return n - 1u;
  return (uint32_t)f;
}

__device__ __forceinline__ uint32_t warp_incl_scan(uint32_t v, int lane) {
#pragma unroll
  for (int d = 1; d < 32; d <<= 1) {
    const uint32_t o = __shfl_up_sync(0xffffffffu, v, d);
    if (lane >= d) v += o;
  }
  return v;
}

// Exclusive scan of one value per thread across the block; returns the exclusive prefix and the
// block total.  `ws` is shared scratch of NT/32 words.
template <int NT>
__device__ __forceinline__ uint32_t block_excl_scan(uint32_t v, uint32_t* ws, uint32_t& total) {
  const int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
  const uint32_t inc = warp_incl_scan(v, lane);
  if (lane == 31) ws[w] = inc;
  __syncthreads();
  uint32_t base = 0, tot = 0;
#pragma unroll
  for (int i = 0; i < NT / 32; ++i) {
    const uint32_t s = ws[i];
    if (i < w) base += s;
    tot += s;
  }
  __syncthreads();
  total = tot;
  return base + inc - v;
}

// ---------------------------------------------------------------------------------------------
// a1 — bin_rows.  One CTA per (sector,row).  The row's clusters are ONE contiguous block of the caller's xyz
// array (12 n bytes): it is read once, with 16-byte loads over its aligned body and scalar loads for the ragged
// head and tail, and staged in shared memory (rows of up to kBinStage clusters; larger rows re-read through L2).
// Then: bin id per cluster + rank inside the bin (shared-memory histogram, arrival order: the order inside a
// bin is not part of the contract, G5), block prefix sum over the bins (warp-shuffle scan), the 16-bit table of
// bin starts, and the scatter of (y, z) and the original index into bin order, all from shared memory.
// HBM traffic: 12 B read, 8 + 4 + 8 B written per cluster (sorted (y,z), original index, cleared owner),
// 2 B per bin; bin_of[] (4 B per cluster) is a debug output that is written once and never read back.
#ifndef TPCST_BIN_STAGE
#define TPCST_BIN_STAGE 1024
#endif
constexpr uint32_t kBinStage = TPCST_BIN_STAGE;                 // clusters of a row staged in shared memory
constexpr uint32_t kBinStageBytes = (3u * kBinStage + 8u) * 4u + kBinStage * 4u;

__global__ void __launch_bounds__(kBlock) bin_rows(const __grid_constant__ Params p) {
  extern __shared__ __align__(16) uint32_t hist[];   // [hist_words] counts, then exclusive starts; then the staging area
  __shared__ uint32_t ws[kBlock / 32];
  if (event_failed(p)) return;
  float* const raw = reinterpret_cast<float*>(hist + p.hist_words);    // [3 n] the row's (x, y, z)
  uint32_t* const code = hist + p.hist_words + 3u * kBinStage + 8u;     // [n] bin | rank inside the bin << 16
  const uint32_t sr = blockIdx.x, k = sr % p.R;
  const uint32_t g0 = p.row_start[sr], g1 = p.row_start[sr + 1];
  const uint32_t n = g1 - g0;
  const RowTab tb = p.tab[k];
  const uint32_t ny = tb.ny, nb = ny * p.nz;
  uint16_t* bins = p.bins + (size_t)(sr / p.R) * p.bins_sector_stride + tb.bin_off;
  const uint32_t sr0 = sr - k;                        // construct_tracklets keeps 16-bit slab offsets (units of kPad) per sector
  // row_start of a TPCST_DEVICE event cannot be validated on the host: monotonicity and its two ends are checked here
  // (the same conditions tpcst_submit_event tests for host input: TPCST_ERR_ARG)
  if (p.n_clusters != 0xffffffffu &&                   // 0xffffffff: host input, validated by tpcst_submit_event
      (g1 < g0 || g1 > p.n_clusters || (sr == 0u && g0 != 0u) || (sr + 1u == gridDim.x && g1 != p.n_clusters))) {
    if (threadIdx.x == 0) atomicOr(&p.ctr->error, kErrArg);
    return;
  }
  if (n > kMaxRowClusters || g1 > p.max_clusters ||
      ((pstart(g0, sr) - pstart(p.row_start[sr0], sr0)) >> 4) > kMaxSectorSlabUnits) {
    if (threadIdx.x == 0) atomicOr(&p.ctr->error, kErrRange);
    return;
  }
  const uint32_t p0 = pstart(g0, sr);
  const bool staged = n <= kBinStage;
  // the per-bin passes (clear, scan, table) work on 16-byte groups: a row has ~6 bins per cluster, and one
  // 32-bit shared-memory instruction per bin and pass kept the shared-memory pipe full (mio_throttle, ncu r01i)
  const uint32_t nb8 = (nb + 1u + 7u) & ~7u;          // entries of the row's table incl. the end marker, padded as in HBM
  uint4* const hist4 = reinterpret_cast<uint4*>(hist);
  for (uint32_t b = threadIdx.x; b < nb8 / 4u; b += kBlock) hist4[b] = make_uint4(0u, 0u, 0u, 0u);
  if (staged) {
    // floats [f0, f1) of xyz: 16-byte loads over [a0, a1), scalar loads for the head and the tail
    const size_t f0 = 3u * (size_t)g0, f1 = 3u * (size_t)g1;
    const bool al16 = (reinterpret_cast<uintptr_t>(p.xyz) & 15u) == 0u;
    const size_t a0 = al16 ? min((f0 + 3u) & ~(size_t)3u, f1) : f1, a1 = al16 ? max(f1 & ~(size_t)3u, a0) : f1;
    for (size_t i = f0 + threadIdx.x; i < a0; i += kBlock) raw[i - f0] = __ldcs(p.xyz + i);
    for (size_t i = a0 + 4u * threadIdx.x; i < a1; i += 4u * kBlock) {
      const float4 v = __ldcs(reinterpret_cast<const float4*>(p.xyz + i));
      float* d = raw + (i - f0);
      d[0] = v.x; d[1] = v.y; d[2] = v.z; d[3] = v.w;
    }
    for (size_t i = a1 + threadIdx.x; i < f1; i += kBlock) raw[i - f0] = __ldcs(p.xyz + i);
  }
  __syncthreads();
  // pass 1: bin id and rank inside the bin
  for (uint32_t i = threadIdx.x; i < n; i += kBlock) {
    float y, z;
    if (staged) { y = raw[3u * i + 1u]; z = raw[3u * i + 2u]; }
    else { y = p.xyz[3 * (size_t)(g0 + i) + 1]; z = p.xyz[3 * (size_t)(g0 + i) + 2]; }
    const uint32_t iy = bin_coord(y, tb.ymax, p.inv_bin_y, ny);
    const uint32_t iz = bin_coord(z, 0.0f, p.inv_bin_z, p.nz);
    const uint32_t b = iz * ny + iy;
    const uint32_t r = atomicAdd(&hist[b], 1u);
    if (staged) code[i] = b | (r << 16);
    p.bin_of[g0 + i] = b | (r << 16);
    owner_clear(p, p0 + i);                          // selection keys start empty
  }
  __syncthreads();
  // exclusive prefix sum over the bins: contiguous chunk of 16-byte groups per thread + block scan of chunk sums
  // (entries [nb, nb8) hold 0 counts, so their starts come out as n: the end marker and the padding)
  const uint32_t ng = nb8 / 4u, chunk = (ng + kBlock - 1) / kBlock;
  const uint32_t b0 = min(threadIdx.x * chunk, ng), b1 = min(b0 + chunk, ng);
  uint32_t s = 0;
  for (uint32_t b = b0; b < b1; ++b) { const uint4 v = hist4[b]; s += (v.x + v.y) + (v.z + v.w); }
  uint32_t total;
  uint32_t run = block_excl_scan<kBlock>(s, ws, total);
  for (uint32_t b = b0; b < b1; ++b) {
    const uint4 v = hist4[b];
    uint4 o;
    o.x = run; o.y = o.x + v.x; o.z = o.y + v.y; o.w = o.z + v.z;
    run = o.w + v.w;
    hist4[b] = o;
  }
  __syncthreads();
  uint4* const bins4 = reinterpret_cast<uint4*>(bins);                  // 8 starts (16 bits each) per 16-byte store
  for (uint32_t b = threadIdx.x; b < nb8 / 8u; b += kBlock) {
    const uint4 lo = hist4[2u * b], hi = hist4[2u * b + 1u];
    bins4[b] = make_uint4(lo.x | (lo.y << 16), lo.z | (lo.w << 16), hi.x | (hi.y << 16), hi.z | (hi.w << 16));
  }
  // pass 2: scatter into bin order
  if (staged) {
    for (uint32_t i = threadIdx.x; i < n; i += kBlock) {
      const uint32_t c = code[i];
      const uint32_t pos = p0 + hist[c & 0xffffu] + (c >> 16);
      p.s_yz[pos] = make_float2(raw[3u * i + 1u], raw[3u * i + 2u]);
      p.s_orig[pos] = g0 + i;
    }
  } else {
    // rows too large to stage: bin and rank come back from bin_of[], the coordinates from L2.  (If the caller's
    // device row_start made two rows overlap, another CTA may have overwritten bin_of: the event has failed by
    // then, and the bounds tests keep this CTA inside its own slab.)
    for (uint32_t i = threadIdx.x; i < n; i += kBlock) {
      const uint32_t br = p.bin_of[g0 + i], b = br & 0xffffu;
      const uint32_t off = (b < nb ? hist[b] : n) + (br >> 16);
      if (off >= n) continue;
      const float y = p.xyz[3 * (size_t)(g0 + i) + 1], z = p.xyz[3 * (size_t)(g0 + i) + 2];
      p.s_yz[p0 + off] = make_float2(y, z);
      p.s_orig[p0 + off] = g0 + i;
    }
  }
}

// ---------------------------------------------------------------------------------------------
// a2 — find_neighbours.  One CTA per (sector,row k), one thread per cluster (L50).  The slabs and
// bin tables of rows k+1 and k-1 are staged in shared memory when they fit (they are contiguous,
// 16-byte aligned runs, copied 16 bytes at a time), else read in place
// through the generic address space.
struct RowSide {
  const float2* yz;      // row-local sorted (y,z)
  const uint16_t* bins;  // ny*nz + 1 exclusive starts
  uint32_t ny, p0;
  float ymax;
};

// D of the pair and the (D, index u, index d) lexicographic comparison of G7/G8.
__device__ __forceinline__ void nf_consider(const Params& p, float y, float z, float t1, float s1, float2 d, float w_dn,
                                            uint32_t qu, uint32_t qd, const RowSide& U, const RowSide& Dn,
                                            float& bestD, int32_t& bu, int32_t& bd) {
  const float t2 = d.x * w_dn;
  const float ey = (t1 + t2) - y;
  const float s2 = d.y * w_dn;
  const float ez = (s1 + s2) - z;
  const float D = (ey * ey) + (ez * ez);
  if (!(D <= p.nf_max_dev2)) return;
  bool take = bu < 0 || D < bestD;
  if (!take && D == bestD) {                          // rare: exact tie -> original indices decide
    const uint32_t ou = p.s_orig[U.p0 + qu], obu = p.s_orig[U.p0 + (uint32_t)bu];
    if (ou < obu) take = true;
    else if (ou == obu) take = p.s_orig[Dn.p0 + qd] < p.s_orig[Dn.p0 + (uint32_t)bd];
  }
  if (take) { bestD = D; bu = (int32_t)qu; bd = (int32_t)qd; }
}

// The nested form of the definition (every down candidate tested for every up candidate inside the
// window): used for clusters whose candidate lists do not fit kNfList entries per side.
template <bool kCount>
__device__ __noinline__ void nf_nested(const Params& p, const RowTab& tb, const RowSide& U, const RowSide& Dn, float y, float z,
                                       float pyu, float pzu, float pyd, float pzd, uint32_t uy0, uint32_t uy1, uint32_t uz0,
                                       uint32_t uz1, uint32_t dy0, uint32_t dy1, uint32_t dz0, uint32_t dz1, float& bestD,
                                       int32_t& bu, int32_t& bd, uint32_t& n_tests, uint32_t& n_pairs) {
  for (uint32_t uz = uz0; uz <= uz1; ++uz) {
    const uint32_t q1 = U.bins[uz * U.ny + uy1 + 1u];
    for (uint32_t qu = U.bins[uz * U.ny + uy0]; qu < q1; ++qu) {
      const float2 u = U.yz[qu];
      const float du = u.x - pyu, dv = u.y - pzu;
      if (!(fabsf(du) <= tb.wy_up) || !(fabsf(dv) <= tb.wz_up)) continue;
      const float t1 = u.x * tb.w_up, s1 = u.y * tb.w_up;        // G7
      for (uint32_t dz = dz0; dz <= dz1; ++dz) {
        const uint32_t r1 = Dn.bins[dz * Dn.ny + dy1 + 1u];
        for (uint32_t qd = Dn.bins[dz * Dn.ny + dy0]; qd < r1; ++qd) {
          const float2 d = Dn.yz[qd];
          const float dd = d.x - pyd, de = d.y - pzd;
          if (!(fabsf(dd) <= tb.wy_dn) || !(fabsf(de) <= tb.wz_dn)) continue;
          if (kCount) ++n_pairs;
          nf_consider(p, y, z, t1, s1, d, tb.w_dn, qu, qd, U, Dn, bestD, bu, bd);
        }
      }
    }
  }
}

template <bool kCount>
__global__ void __launch_bounds__(kBlock) find_neighbours(const __grid_constant__ Params p) {
  extern __shared__ __align__(16) unsigned char smem_raw[];
  __shared__ uint16_t nf_list[2 * kNfList * kBlock];  // [side][slot][thread] candidate lists
  uint32_t n_tests = 0, n_pairs = 0;                  // work counters (kCount only)
  if (event_failed(p)) return;
  const uint32_t sr = blockIdx.x, k = sr % p.R, sec = sr / p.R;
  const uint32_t g0 = p.row_start[sr], n = p.row_start[sr + 1] - g0;
  const uint32_t p0 = pstart(g0, sr);
  if (k == 0 || k + 1 >= p.R) {                       // G9
    for (uint32_t i = threadIdx.x; i < n; i += kBlock) { p.up_raw[p0 + i] = -1; p.dn_raw[p0 + i] = -1; }
    return;
  }
  const RowTab tb = p.tab[k], tu = p.tab[k + 1], td = p.tab[k - 1];
  const uint32_t gu = p.row_start[sr + 1], nu = p.row_start[sr + 2] - gu;
  const uint32_t gd = p.row_start[sr - 1], nd = g0 - gd;
  RowSide U, Dn;
  U.p0 = pstart(gu, sr + 1); Dn.p0 = pstart(gd, sr - 1);
  U.ny = tu.ny; Dn.ny = td.ny; U.ymax = tu.ymax; Dn.ymax = td.ymax;
  const uint16_t* gbu = p.bins + (size_t)sec * p.bins_sector_stride + tu.bin_off;
  const uint16_t* gbd = p.bins + (size_t)sec * p.bins_sector_stride + td.bin_off;
  const uint32_t nbu = tu.ny * p.nz + 1u, nbd = td.ny * p.nz + 1u;
  // shared-memory plan (all pieces 16-byte multiples)
  const uint32_t byu = ((nu * 8u) + 15u) & ~15u, byd = ((nd * 8u) + 15u) & ~15u;
  const uint32_t bbu = ((nbu * 2u) + 15u) & ~15u, bbd = ((nbd * 2u) + 15u) & ~15u;
  if (byu + byd + bbu + bbd <= p.nf_smem_bytes) {
    // The four pieces are contiguous, 16-byte aligned runs of HBM: plain 16-byte copies by all threads, through L1
    // (the slab of a row is staged by the CTAs of both its neighbours, often on the same SM).  TMA bulk copies
    // (cp.async.bulk completing on an mbarrier) were built and measured in round 1: the kernel
    // alone 0.210 ms against 0.220 ms, but the pipelined event stream 589 against 611 events/s, because the bulk
    // copies always go to L2, which the other events' selection kernels are bound by.  That path was removed.
    {
      uint4* d4 = reinterpret_cast<uint4*>(smem_raw);
      const uint4* s0 = reinterpret_cast<const uint4*>(p.s_yz + U.p0);
      const uint4* s1 = reinterpret_cast<const uint4*>(p.s_yz + Dn.p0);
      const uint4* s2 = reinterpret_cast<const uint4*>(gbu);
      const uint4* s3 = reinterpret_cast<const uint4*>(gbd);
      const uint32_t c0 = byu / 16, c1 = byd / 16, c2 = bbu / 16, c3 = bbd / 16;
      for (uint32_t i = threadIdx.x; i < c0; i += kBlock) d4[i] = s0[i];
      for (uint32_t i = threadIdx.x; i < c1; i += kBlock) d4[c0 + i] = s1[i];
      for (uint32_t i = threadIdx.x; i < c2; i += kBlock) d4[c0 + c1 + i] = s2[i];
      for (uint32_t i = threadIdx.x; i < c3; i += kBlock) d4[c0 + c1 + c2 + i] = s3[i];
    }
    U.yz = reinterpret_cast<const float2*>(smem_raw);
    Dn.yz = reinterpret_cast<const float2*>(smem_raw + byu);
    U.bins = reinterpret_cast<const uint16_t*>(smem_raw + byu + byd);
    Dn.bins = reinterpret_cast<const uint16_t*>(smem_raw + byu + byd + bbu);
    __syncthreads();
  } else {
    U.yz = p.s_yz + U.p0; Dn.yz = p.s_yz + Dn.p0; U.bins = gbu; Dn.bins = gbd;
  }
  // Two phases per cluster.  (1) The clusters of row k+1 inside the up window and those of row k-1
  // inside the down window are collected (row-local indices, up to kNfList per side, in shared
  // memory, slot-major = conflict-free).  (2) The |U| x |D| pairs are evaluated in one flat loop.
  // The window predicate of a down candidate does not depend on the up candidate, so this does
  // nu + nd window tests and |U||D| pair evaluations where the nested form of the definition does
  // nu + |U| nd, and the warp's loops are as long as its longest list, not its longest product.
  // A cluster with more than kNfList candidates on a side takes the nested form (same result).
  uint16_t* const lu = nf_list + threadIdx.x;
  uint16_t* const ld = nf_list + kNfList * kBlock + threadIdx.x;
  for (uint32_t i = threadIdx.x; i < n; i += kBlock) {
    const float2 c = p.s_yz[p0 + i];
    const float y = c.x, z = c.y;
    const float pyu = y * tb.ratio_up, pzu = z * tb.ratio_up;        // G6
    const float pyd = y * tb.ratio_dn, pzd = z * tb.ratio_dn;
    float bestD = 0.0f;
    int32_t bu = -1, bd = -1;
    if (nu != 0u && nd != 0u) {
      const uint32_t uy0 = bin_coord((pyu - tb.wy_up) - p.grid_pad, U.ymax, p.inv_bin_y, U.ny);
      const uint32_t uy1 = bin_coord((pyu + tb.wy_up) + p.grid_pad, U.ymax, p.inv_bin_y, U.ny);
      const uint32_t uz0 = bin_coord((pzu - tb.wz_up) - p.grid_pad, 0.0f, p.inv_bin_z, p.nz);
      const uint32_t uz1 = bin_coord((pzu + tb.wz_up) + p.grid_pad, 0.0f, p.inv_bin_z, p.nz);
      const uint32_t dy0 = bin_coord((pyd - tb.wy_dn) - p.grid_pad, Dn.ymax, p.inv_bin_y, Dn.ny);
      const uint32_t dy1 = bin_coord((pyd + tb.wy_dn) + p.grid_pad, Dn.ymax, p.inv_bin_y, Dn.ny);
      const uint32_t dz0 = bin_coord((pzd - tb.wz_dn) - p.grid_pad, 0.0f, p.inv_bin_z, p.nz);
      const uint32_t dz1 = bin_coord((pzd + tb.wz_dn) + p.grid_pad, 0.0f, p.inv_bin_z, p.nz);
      // candidates of a window = (at most) two contiguous runs of the slab, walked as one flat loop
      uint32_t cu = 0u, cd = 0u;
      bool nested = uz1 > uz0 + 1u || dz1 > dz0 + 1u;     // a window higher than two grid rows: rare
      if (!nested) {
        const uint32_t ub = uz0 * U.ny;
        const uint32_t qa = U.bins[ub + uy0], qb = U.bins[ub + uy1 + 1u];
        uint32_t ra = 0u, rb = 0u;
        if (uz1 > uz0) { ra = U.bins[ub + U.ny + uy0]; rb = U.bins[ub + U.ny + uy1 + 1u]; }
        const uint32_t n0 = qb - qa, nn = n0 + (rb - ra), off1 = ra - n0;
        if (kCount) n_tests += nn;
        for (uint32_t j = 0; j < nn; ++j) {
          const uint32_t qu = (j < n0 ? qa : off1) + j;
          const float2 u = U.yz[qu];
          const bool pass = fabsf(u.x - pyu) <= tb.wy_up && fabsf(u.y - pzu) <= tb.wz_up;
          if (pass && cu < kNfList) lu[cu * kBlock] = (uint16_t)qu;
          cu += pass ? 1u : 0u;
        }
      }
      if (!nested && cu != 0u) {
        const uint32_t db = dz0 * Dn.ny;
        const uint32_t qa = Dn.bins[db + dy0], qb = Dn.bins[db + dy1 + 1u];
        uint32_t ra = 0u, rb = 0u;
        if (dz1 > dz0) { ra = Dn.bins[db + Dn.ny + dy0]; rb = Dn.bins[db + Dn.ny + dy1 + 1u]; }
        const uint32_t n0 = qb - qa, nn = n0 + (rb - ra), off1 = ra - n0;
        if (kCount) n_tests += nn;
        for (uint32_t j = 0; j < nn; ++j) {
          const uint32_t qd = (j < n0 ? qa : off1) + j;
          const float2 d = Dn.yz[qd];
          const bool pass = fabsf(d.x - pyd) <= tb.wy_dn && fabsf(d.y - pzd) <= tb.wz_dn;
          if (pass && cd < kNfList) ld[cd * kBlock] = (uint16_t)qd;
          cd += pass ? 1u : 0u;
        }
      }
      nested = nested || cu > kNfList || cd > kNfList;
      if (!nested) {
        // D >= 0, so its bit pattern orders like its value: the minimum is an unsigned compare; an exact
        // tie of the minimum (rare) is settled by the nested form with its index comparisons (G8)
        const uint32_t np = cu * cd;
        if (kCount) n_pairs += np;
        uint32_t iu = 0u, id = 0u, bkey = 0xffffffffu;
        bool tie = false;
        for (uint32_t pi = 0; pi < np; ++pi) {
          const uint32_t qu = lu[iu * kBlock], qd = ld[id * kBlock];
          const float2 u = U.yz[qu], d = Dn.yz[qd];
          const float ey = (u.x * tb.w_up + d.x * tb.w_dn) - y;       // G7
          const float ez = (u.y * tb.w_up + d.y * tb.w_dn) - z;
          const float D = (ey * ey) + (ez * ez);
          const uint32_t key = D <= p.nf_max_dev2 ? __float_as_uint(D) : 0xffffffffu;
          tie = tie || key == bkey;
          if (key < bkey) { bkey = key; bu = (int32_t)qu; bd = (int32_t)qd; tie = false; }
          if (++id == cd) { id = 0u; ++iu; }
        }
        if (bkey == 0xffffffffu) bu = -1;
        nested = tie && bkey != 0xffffffffu;
        if (nested) { uint32_t t0 = 0u, t1 = 0u; bu = -1; bd = -1;
          nf_nested<false>(p, tb, U, Dn, y, z, pyu, pzu, pyd, pzd, uy0, uy1, uz0, uz1, dy0, dy1, dz0, dz1, bestD, bu, bd, t0, t1); }
      } else {
        nf_nested<kCount>(p, tb, U, Dn, y, z, pyu, pzu, pyd, pzd, uy0, uy1, uz0, uz1, dy0, dy1, dz0, dz1, bestD, bu, bd, n_tests, n_pairs);
      }
    }
    p.up_raw[p0 + i] = bu >= 0 ? (int32_t)(U.p0 + (uint32_t)bu) : -1;
    p.dn_raw[p0 + i] = bu >= 0 ? (int32_t)(Dn.p0 + (uint32_t)bd) : -1;
  }
  if (kCount) {
    __syncwarp();
    count_add_warp(&p.ctr->nf_window_tests, n_tests);
    count_add_warp(&p.ctr->nf_pair_evals, n_pairs);
  }
}

// ---------------------------------------------------------------------------------------------
// a3 — evolve_links: keep reciprocal links only (L41).  Streaming pass over the row's links with
// one gather per link, out of place so the raw links stay available to the parity tests.
__global__ void __launch_bounds__(kBlock) evolve_links(const __grid_constant__ Params p) {
  if (event_failed(p)) return;
  const uint32_t sr = blockIdx.x;
  const uint32_t g0 = p.row_start[sr], n = p.row_start[sr + 1] - g0;
  const uint32_t p0 = pstart(g0, sr);
  for (uint32_t i = threadIdx.x; i < n; i += kBlock) {
    const int32_t pos = (int32_t)(p0 + i);
    const int32_t u = p.up_raw[pos], d = p.dn_raw[pos];
    p.up[pos] = (u >= 0 && p.dn_raw[u] == pos) ? u : -1;
    p.dn[pos] = (d >= 0 && p.up_raw[d] == pos) ? d : -1;
  }
}

// ---------------------------------------------------------------------------------------------
// a4 — find_starts: start = up link, no down link (G12); chain followed for min_chain clusters; kept
// starts are compacted per row in ORIGINAL-index order so that tracklet ids do not depend on the
// (arbitrary) order inside a grid bin.
__global__ void __launch_bounds__(kBlock) find_starts(const __grid_constant__ Params p) {
  __shared__ uint32_t ws[kBlock / 32];
  if (event_failed(p)) return;
  const uint32_t sr = blockIdx.x;
  const uint32_t g0 = p.row_start[sr], n = p.row_start[sr + 1] - g0;
  const uint32_t p0 = pstart(g0, sr);
  for (uint32_t i = threadIdx.x; i < n; i += kBlock) {
    const uint32_t pos = p0 + i;
    uint32_t mark = 0u;
    int32_t c = p.up[pos];
    if (c >= 0 && p.dn[pos] < 0) {                     // G12; only "length >= min_chain" is needed here,
      uint32_t len = 1u;                                // so the walk stops there (the full chain is
      for (; c >= 0 && len < p.min_chain; c = p.up[c]) ++len;   // followed by construct_tracklets)
      if (len >= p.min_chain) mark = i + 1u;
    }
    p.start_mark[p.s_orig[pos]] = mark;
  }
  __syncthreads();
  uint32_t base = 0u;
  for (uint32_t i0 = 0; i0 < n; i0 += kBlock) {      // ordered compaction, tile by tile
    const uint32_t i = i0 + threadIdx.x;
    const uint32_t m = i < n ? p.start_mark[g0 + i] : 0u;
    uint32_t total;
    const uint32_t r = block_excl_scan<kBlock>(m != 0u ? 1u : 0u, ws, total);
    if (m != 0u) p.start_list[p0 + base + r] = p0 + m - 1u;
    base += total;
  }
  if (threadIdx.x == 0) p.row_cnt[sr] = base;
}

// Exclusive scan of the per-row start counts -> first tracklet id of every row; total -> counters.
// (Tracklet ids follow (sector, row, original index) order: DESIGN.md G12.)  A second CTA scans the
// same counts in (row, sector) order: the offsets of the work list (list_tracklets).
__global__ void __launch_bounds__(1024) scan_rows(const __grid_constant__ Params p) {
  __shared__ uint32_t ws[32];
  if (event_failed(p)) return;
  const uint32_t SR = p.S * p.R;
  const bool by_row = blockIdx.x == 1u;               // CTA 0: (sector,row) order; CTA 1: (row,sector) order
  uint32_t* const out = by_row ? p.ord_off : p.row_off;
  // every thread owns a contiguous chunk (two passes over it); the chunk sums are scanned across the block
  const uint32_t chunk = (SR + 1023u) / 1024u, i0 = min(threadIdx.x * chunk, SR), i1 = min(i0 + chunk, SR);
  auto src = [&](uint32_t i) { if (!by_row) return i; const uint32_t k = i / p.S; return (i - k * p.S) * p.R + k; };
  uint32_t sum = 0u;
  for (uint32_t i = i0; i < i1; ++i) sum += p.row_cnt[src(i)];
  uint32_t total;
  uint32_t run = block_excl_scan<1024>(sum, ws, total);
  for (uint32_t i = i0; i < i1; ++i) { out[i] = run; run += p.row_cnt[src(i)]; }
  if (threadIdx.x == 0) {
    out[SR] = total;
    if (!by_row) {
      if (total > p.tcap) { atomicOr(&p.ctr->error, kErrTrackletCap); total = 0u; }
      p.ctr->n_tracklets = total;
    }
  }
}

cudaError_t configure_ca(uint32_t hist_words, uint32_t nf_bytes, uint32_t* bin_rows_smem_bytes) {
  *bin_rows_smem_bytes = hist_words * 4u + kBinStageBytes;
  cudaError_t e = cudaFuncSetAttribute(bin_rows, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)*bin_rows_smem_bytes);
  if (e != cudaSuccess) return e;
  e = cudaFuncSetAttribute(find_neighbours<false>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)nf_bytes);
  if (e != cudaSuccess) return e;
  return cudaFuncSetAttribute(find_neighbours<true>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)nf_bytes);
}

void launch_ca(const Params& p, cudaStream_t st, cudaEvent_t* ev, bool count) {
  const uint32_t SR = p.S * p.R;
  bin_rows<<<SR, kBlock, p.hist_smem_bytes, st>>>(p);        mark(ev, 0, st);
  if (count) find_neighbours<true><<<SR, kBlock, p.nf_smem_bytes, st>>>(p);
  else find_neighbours<false><<<SR, kBlock, p.nf_smem_bytes, st>>>(p);
  mark(ev, 1, st);
  evolve_links<<<SR, kBlock, 0, st>>>(p);                    mark(ev, 2, st);
  find_starts<<<SR, kBlock, 0, st>>>(p);                     mark(ev, 3, st);
  scan_rows<<<2, 1024, 0, st>>>(p);                          mark(ev, 4, st);
}

}  // namespace tpcst
