// tpcca_links.cu -- steps (b) neighbours finder, (c) neighbours cleaner, (d) start-hit finder.
// (b) PAPER.md:49 "links between hit triplets arranged close to a straight line", parallel over hits
//     (PAPER.md:57), window centred on the hit, no vertex constraint.  DESIGN.md O2.
// (c) mutual links only (north_star (c); O3).  (d) chain heads, canonical order (O4).
#include "tpcca_dev.cuh"

// ---------------------------------------------------------------- (b)
// One thread per sorted cluster; consecutive threads are neighbours in (row, y-bin, z-bin), so a warp's
// candidate ranges overlap (L1 hits) and its loop trip counts are close.  Three phases keep the lanes together:
// the window candidates of the down row and of the up row are collected into per-thread shared-memory lists
// (NB_CAP entries each; the bins of up to two y-bin rows form one flat index space walked NB_UNROLL at a time
// with independent loads), then the (up, down) pairs are evaluated from shared memory.  A list that overflows
// (dense noise) falls back to the plain nested loops -- same result either way.
#ifndef NB_THREADS
#define NB_THREADS 64
#endif
#ifndef NB_CAP
#define NB_CAP 7
#endif
#ifndef NB_UNROLL
#define NB_UNROLL 2
#endif
#ifndef NB_MINBLOCKS
#define NB_MINBLOCKS 20
#endif

struct Best {
  int bu, bd;
  float bc;
};

// (plain pointers, not Dev&: a reference to the kernel parameter block would force a local-memory copy of it)
__device__ __noinline__ bool pair_tie_better(const float2* yz, const int32_t* orig_idx, int bu, int bd, int u, float yu,
                                             float zu, int dd, float yd, float zd) {
  if (u != bu) {
    const float2 q = yz[bu];
    return key_less(zu, yu, orig_idx[u], q.y, q.x, orig_idx[bu]);
  }
  const float2 q = yz[bd];
  return key_less(zd, yd, orig_idx[dd], q.y, q.x, orig_idx[bd]);
}

__device__ __forceinline__ void consider(const Dev& d, Best& b, float cost, int u, float yu, float zu, int dd, float yd,
                                         float zd) {
  if (!(cost <= d.P.triplet_cut)) return;
  bool better = (b.bu < 0) || (cost < b.bc);
  if (!better && cost == b.bc) better = pair_tie_better(d.yz, d.orig_idx, b.bu, b.bd, u, yu, zu, dd, yd, zd);  // exact tie: key order (rare)
  if (better) { b.bu = u; b.bd = dd; b.bc = cost; }
}

// Window candidates of one neighbour row: appended to the calling thread's shared-memory list; returns their number
// (entries beyond NB_CAP are counted, not stored).  The bins of up to two y-bin rows form one flat index space
// [0, ntot): index i < na is cluster a0 + i, the others b0 + (i - na); the body is predicated, not branched.
__device__ __forceinline__ int collect(const Dev& d, const GridHdr& g, float y0, float z0, float wy, float wz, float mz,
                                       float2* __restrict__ lp, int* __restrict__ li) {
  int by0, by1, bz0, bz1;
  bin_range_fast(y0 - wy - 1e-3f, y0 + wy + 1e-3f, g.ymin, g.inv_by, g.ny, by0, by1);
  bin_range_fast(z0 - wz - mz, z0 + wz + mz, g.zmin, g.inv_bz, g.nz, bz0, bz1);
  if (bz0 > bz1) return 0;
  int n = 0;
  for (int by = by0; by <= by1; by += 2) {
    const int* bs = d.bin_start + g.bin_base + by * g.nz;
    const int a0 = bs[bz0], a1 = bs[bz1 + 1];
    int b0 = 0, b1 = 0;
    if (by + 1 <= by1) { b0 = bs[g.nz + bz0]; b1 = bs[g.nz + bz1 + 1]; }
    const int na = a1 - a0, ntot = na + (b1 - b0);
    const int jump = b0 - a1;  // index i >= na is cluster a0 + i + jump
    for (int i = 0; i < ntot; i += NB_UNROLL) {
      float2 p[NB_UNROLL];
      int c[NB_UNROLL];
#pragma unroll
      for (int j = 0; j < NB_UNROLL; j++) {
        const int ii = min(i + j, ntot - 1);
        c[j] = a0 + ii + ((ii >= na) ? jump : 0);
        p[j] = d.yz[c[j]];
      }
#pragma unroll
      for (int j = 0; j < NB_UNROLL; j++) {
        const bool in = (i + j < ntot) && (fabsf(p[j].x - y0) <= wy) && (fabsf(p[j].y - z0) <= wz);
        if (in) {
          const int slot = min(n, NB_CAP - 1) * NB_THREADS;  // an overflowing list is never read (fallback path)
          lp[slot] = p[j];
          li[slot] = c[j];
        }
        n += in ? 1 : 0;
      }
    }
  }
  return n;
}

// Fallback for overflowing lists: plain nested loops over both windows (O2 as written).
__device__ __forceinline__ void nested_pairs(const Dev& d, const NbrHdr& nb, const GridHdr& gu, const GridHdr& gd, float y0,
                                          float z0, float mz, Best& best) {
  int uy0, uy1, uz0, uz1, dy0, dy1, dz0, dz1;
  bin_range(y0 - nb.wyu - 1e-3f, y0 + nb.wyu + 1e-3f, gu.ymin, gu.inv_by, gu.ny, uy0, uy1);
  bin_range(z0 - nb.wzu - mz, z0 + nb.wzu + mz, gu.zmin, gu.inv_bz, gu.nz, uz0, uz1);
  bin_range(y0 - nb.wyd - 1e-3f, y0 + nb.wyd + 1e-3f, gd.ymin, gd.inv_by, gd.ny, dy0, dy1);
  bin_range(z0 - nb.wzd - mz, z0 + nb.wzd + mz, gd.zmin, gd.inv_bz, gd.nz, dz0, dz1);
  if (uz0 > uz1 || dz0 > dz1) return;
  const float t = nb.t;
  for (int by = uy0; by <= uy1; by++) {
    const int* bs = d.bin_start + gu.bin_base + by * gu.nz;
    const int ub = bs[uz0], ue = bs[uz1 + 1];
    for (int u = ub; u < ue; u++) {
      const float2 pu = d.yz[u];
      if (!(fabsf(pu.x - y0) <= nb.wyu) || !(fabsf(pu.y - z0) <= nb.wzu)) continue;
      for (int by2 = dy0; by2 <= dy1; by2++) {
        const int* bs2 = d.bin_start + gd.bin_base + by2 * gd.nz;
        const int db = bs2[dz0], de = bs2[dz1 + 1];
        for (int dd = db; dd < de; dd++) {
          const float2 pd = d.yz[dd];
          if (!(fabsf(pd.x - y0) <= nb.wyd) || !(fabsf(pd.y - z0) <= nb.wzd)) continue;
          const float ey = y0 - fmaf(t, pu.x - pd.x, pd.x);
          const float ez = z0 - fmaf(t, pu.y - pd.y, pd.y);
          const float cost = fmaf(ez * ez, d.inv_sz2, (ey * ey) * d.inv_sy2);
          consider(d, best, cost, u, pu.x, pu.y, dd, pd.x, pd.y);
        }
      }
    }
  }
}

// Warp-cooperative path for a cluster whose candidate lists overflowed (dense rows): the 32 lanes of the warp scan the
// window of lane `src` together (lanes stride over the clusters of each y-bin row, a ballot compacts the ones inside the
// window into the warp's part of the shared-memory lists, which the per-thread phase no longer needs), then share the
// nu x nd pairs and reduce to the minimum by (cost, key(u), key(d)).  Without it the one overflowing lane walked the
// nested loops alone while 31 lanes waited (0.16 of 0.86 ms on the 15 M-cluster frame).  Returns false if a window holds
// more than NB_WCAP clusters (the caller then takes the serial nested loops); the result is valid in every lane.
#define NB_WCAP (NB_CAP * 32)
#define FULLW 0xffffffffu
__device__ __forceinline__ int coop_collect(const Dev& d, const GridHdr& g, float y0, float z0, float wy, float wz, float mz,
                                            float2 (*sp)[NB_THREADS], int (*si)[NB_THREADS], int wbase, int lane) {
  int by0, by1, bz0, bz1;
  bin_range(y0 - wy - 1e-3f, y0 + wy + 1e-3f, g.ymin, g.inv_by, g.ny, by0, by1);
  bin_range(z0 - wz - mz, z0 + wz + mz, g.zmin, g.inv_bz, g.nz, bz0, bz1);
  if (bz0 > bz1) return 0;
  int n = 0;
  for (int by = by0; by <= by1; by++) {
    const int* bs = d.bin_start + g.bin_base + by * g.nz;
    const int a0 = bs[bz0], a1 = bs[bz1 + 1];
    for (int c0 = a0; c0 < a1; c0 += 32) {
      const int c = c0 + lane;
      float2 p = make_float2(0.f, 0.f);
      bool in = false;
      if (c < a1) {
        p = d.yz[c];
        in = (fabsf(p.x - y0) <= wy) && (fabsf(p.y - z0) <= wz);
      }
      const unsigned m = __ballot_sync(FULLW, in);
      const int k = n + __popc(m & ((1u << lane) - 1u));
      if (in && k < NB_WCAP) { sp[k >> 5][wbase + (k & 31)] = p; si[k >> 5][wbase + (k & 31)] = c; }
      n += __popc(m);
    }
  }
  return n;
}

__device__ __forceinline__ bool coop_pairs(const Dev& d, int src, float y0, float z0, float mz, const NbrHdr& nb, const GridHdr& gu,
                                        const GridHdr& gd, float2 (*sp)[NB_CAP][NB_THREADS], int (*si)[NB_CAP][NB_THREADS],
                                        Best& out) {
  const int lane = threadIdx.x & 31, wbase = threadIdx.x & ~31;
  __syncwarp();
  const int nd = coop_collect(d, gd, y0, z0, nb.wyd, nb.wzd, mz, sp[0], si[0], wbase, lane);
  const int nu = coop_collect(d, gu, y0, z0, nb.wyu, nb.wzu, mz, sp[1], si[1], wbase, lane);
  if (nd > NB_WCAP || nu > NB_WCAP) return false;
  __syncwarp();
  Best b;
  b.bu = -1; b.bd = -1; b.bc = 0.0f;
  float bzu = 0.f, byu = 0.f, bzd = 0.f, byd = 0.f;  // coordinates of the lane's best pair (tie order)
  const float t = nb.t;
  const int np = nu * nd;
  for (int q = lane; q < np; q += 32) {
    const int ju = q / nd, jd = q - ju * nd;
    const float2 pu = sp[1][ju >> 5][wbase + (ju & 31)], pd = sp[0][jd >> 5][wbase + (jd & 31)];
    const int u = si[1][ju >> 5][wbase + (ju & 31)], dd = si[0][jd >> 5][wbase + (jd & 31)];
    const float ey = y0 - fmaf(t, pu.x - pd.x, pd.x);
    const float ez = z0 - fmaf(t, pu.y - pd.y, pd.y);
    const float cost = fmaf(ez * ez, d.inv_sz2, (ey * ey) * d.inv_sy2);
    if (!(cost <= d.P.triplet_cut)) continue;
    bool better = (b.bu < 0) || (cost < b.bc);
    if (!better && cost == b.bc) {
      if (u != b.bu) better = key_less(pu.y, pu.x, d.orig_idx[u], bzu, byu, d.orig_idx[b.bu]);
      else better = key_less(pd.y, pd.x, d.orig_idx[dd], bzd, byd, d.orig_idx[b.bd]);
    }
    if (better) { b.bu = u; b.bd = dd; b.bc = cost; bzu = pu.y; byu = pu.x; bzd = pd.y; byd = pd.x; }
  }
  // warp minimum by (cost, key(u), key(d)); lanes without a pair lose
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) {
    const int ou = __shfl_xor_sync(FULLW, b.bu, o), od = __shfl_xor_sync(FULLW, b.bd, o);
    const float oc = __shfl_xor_sync(FULLW, b.bc, o);
    const float ozu = __shfl_xor_sync(FULLW, bzu, o), oyu = __shfl_xor_sync(FULLW, byu, o);
    const float ozd = __shfl_xor_sync(FULLW, bzd, o), oyd = __shfl_xor_sync(FULLW, byd, o);
    bool take = false;
    if (ou >= 0) {
      if (b.bu < 0 || oc < b.bc) take = true;
      else if (oc == b.bc) {
        if (ou != b.bu) take = key_less(ozu, oyu, d.orig_idx[ou], bzu, byu, d.orig_idx[b.bu]);
        else if (od != b.bd) take = key_less(ozd, oyd, d.orig_idx[od], bzd, byd, d.orig_idx[b.bd]);
      }
    }
    if (take) { b.bu = ou; b.bd = od; b.bc = oc; bzu = ozu; byu = oyu; bzd = ozd; byd = oyd; }
  }
  out = b;
  (void)src;
  return true;
}

__global__ void __launch_bounds__(NB_THREADS, NB_MINBLOCKS) k_neighbours(Dev d) {
  __shared__ float2 s_p[2][NB_CAP][NB_THREADS];
  __shared__ int s_i[2][NB_CAP][NB_THREADS];
  const int h = blockIdx.x * NB_THREADS + threadIdx.x;
  const bool live = h < d.row_start[d.n_slices];
  if (__ballot_sync(FULLW, live) == 0u) return;  // lanes past the end stay for the warp-cooperative phase
  const int sl = live ? d.slice_of[h] : 0;
  NbrHdr nb = d.nbr[sl];
  if (!live) nb.su = -1;
  Best best;
  best.bu = -1; best.bd = -1; best.bc = 0.0f;
  bool overflow = false;
  float y0 = 0.f, z0 = 0.f, mz = 0.f;
  if (nb.su >= 0) {
    const float2 p0 = d.yz[h];
    y0 = p0.x; z0 = p0.y;
    mz = 1e-3f + fabsf(z0) * 4e-7f;
    const GridHdr gd = d.grid[nb.sd];
    float2* lpd = &s_p[0][0][threadIdx.x];
    int* lid = &s_i[0][0][threadIdx.x];
    const int nd = collect(d, gd, y0, z0, nb.wyd, nb.wzd, mz, lpd, lid);
    if (nd > 0) {
      const GridHdr gu = d.grid[nb.su];
      float2* lpu = &s_p[1][0][threadIdx.x];
      int* liu = &s_i[1][0][threadIdx.x];
      const int nu = collect(d, gu, y0, z0, nb.wyu, nb.wzu, mz, lpu, liu);
      if (nd <= NB_CAP && nu <= NB_CAP) {
        const float t = nb.t;
        // One flat loop over the nu x nd pairs, lanes with different list shapes stay together; the body is
        // branch-free (selects) apart from the exact-tie test, which is rare.  The best pair is tracked by its list
        // positions; min by (cost, key(u), key(d)) among cost <= triplet_cut (O2).
        const int np = nu * nd;
        int ju = 0, jd = 0, bju = -1, bjd = 0;
        float bc = d.P.triplet_cut;
        float2 pu = lpu[0];
        for (int q = 0; q < np; q++) {
          const float2 pd = lpd[jd * NB_THREADS];
          const float ey = y0 - fmaf(t, pu.x - pd.x, pd.x);
          const float ez = z0 - fmaf(t, pu.y - pd.y, pd.y);
          const float cost = fmaf(ez * ez, d.inv_sz2, (ey * ey) * d.inv_sy2);
          bool take = cost < bc;
          if (cost == bc) {  // cost == triplet_cut with no pair yet, or an exact tie between two pairs
            take = bju < 0;
            if (!take) {
              const float2 qu = lpu[bju * NB_THREADS], qd = lpd[bjd * NB_THREADS];
              const int u = liu[ju * NB_THREADS], bu = liu[bju * NB_THREADS];
              if (u != bu) take = key_less(pu.y, pu.x, d.orig_idx[u], qu.y, qu.x, d.orig_idx[bu]);
              else take = key_less(pd.y, pd.x, d.orig_idx[lid[jd * NB_THREADS]], qd.y, qd.x, d.orig_idx[lid[bjd * NB_THREADS]]);
            }
          }
          bju = take ? ju : bju;
          bjd = take ? jd : bjd;
          bc = take ? cost : bc;
          const bool wrap = (jd + 1 == nd);
          jd = wrap ? 0 : jd + 1;
          ju = wrap ? min(ju + 1, NB_CAP - 1) : ju;
          if (wrap) pu = lpu[ju * NB_THREADS];
        }
        if (bju >= 0) { best.bu = liu[bju * NB_THREADS]; best.bd = lid[bjd * NB_THREADS]; best.bc = bc; }
      } else if (nu > 0) {
        overflow = true;
      }
    }
  }
  // clusters whose lists overflowed: one at a time, by the whole warp
  unsigned todo = __ballot_sync(FULLW, overflow);
  while (todo) {
    const int src = __ffs(todo) - 1;
    todo &= todo - 1;
    const int ssl = __shfl_sync(FULLW, sl, src);
    const float sy = __shfl_sync(FULLW, y0, src), sz = __shfl_sync(FULLW, z0, src), smz = __shfl_sync(FULLW, mz, src);
    const NbrHdr snb = d.nbr[ssl];
    const GridHdr gu = d.grid[snb.su], gd = d.grid[snb.sd];
    Best b;
    const bool ok = coop_pairs(d, src, sy, sz, smz, snb, gu, gd, s_p, s_i, b);
    if ((threadIdx.x & 31) == src) {
      if (ok) best = b;
      else nested_pairs(d, snb, gu, gd, sy, sz, smz, best);
    }
  }
  if (live) {
    d.link_up[h] = best.bu;
    d.link_down[h] = best.bd;
  }
}

void launch_neighbours(const Dev& d, Launch& L) {
  if (d.n <= 0) return;
  KTIMED(L, TPCCA_K_NEIGHBOURS, (k_neighbours<<<(d.n + NB_THREADS - 1) / NB_THREADS, NB_THREADS, 0, L.st>>>(d)));
  L.count++;
}

// ---------------------------------------------------------------- (c) + (d1)
// Out-of-place cleaning (raw links stay available for the parity export), start flags, per-slice start
// counts and an arrival-order list of the start hits (one global atomic per block).
__global__ void __launch_bounds__(256) k_clean(Dev d) {
  __shared__ int sm[32];
  __shared__ int s_base;
  const int h = blockIdx.x * blockDim.x + threadIdx.x;
  bool start = false;
  if (h < d.row_start[d.n_slices]) {
    int u = d.link_up[h], dn = d.link_down[h];
    if (u >= 0 && d.link_down[u] != h) u = -1;
    if (dn >= 0 && d.link_up[dn] != h) dn = -1;
    d.link_up_clean[h] = u;
    d.shared_flag[h] = 0;
    start = (dn < 0) && (u >= 0);
    if (start) atomicAdd(&d.slice_nstart[d.slice_of[h]], 1);
  }
  int tot;
  const int e = block_scan_excl(start ? 1 : 0, &tot, sm);
  if (tot == 0) return;
  if (threadIdx.x == 0) s_base = atomicAdd(&d.cnt->n_start_raw, tot);
  __syncthreads();
  if (start) {
    d.start_tmp[s_base + e] = h;
  }
}

// (d2) exclusive scan of per-slice start counts; capacity keeps whole slices only (lowest ids kept)
__global__ void __launch_bounds__(1024) k_start_offsets(Dev d) {
  __shared__ int sm[32];
  __shared__ int s_keep;
  if (threadIdx.x == 0) s_keep = 0;
  __syncthreads();
  int carry = 0;
  for (int b0 = 0; b0 < d.n_slices; b0 += 1024) {
    const int sl = b0 + threadIdx.x;
    const int v = (sl < d.n_slices) ? d.slice_nstart[sl] : 0;
    int tot;
    const int e = block_scan_excl(v, &tot, sm);
    if (sl < d.n_slices) {
      d.slice_sbase[sl] = carry + e;
      if (carry + e + v <= d.max_tracklets) atomicMax(&s_keep, carry + e + v);
    }
    carry += tot;
  }
  __syncthreads();
  if (threadIdx.x == 0) {
    d.slice_sbase[d.n_slices] = carry;
    if (carry > d.max_tracklets) atomicOr(&d.cnt->status, TPCCA_STAT_TRACKLET_OVERFLOW);
    d.cnt->n_start = (carry <= d.max_tracklets) ? carry : s_keep;
  }
}

// (d3) canonical order = (slice, ord z, ord y, input index).  Bucket sort: every slice with m start hits
// owns m z-buckets (monotone in z) at [slice_sbase, slice_sbase+m); a global scan of the bucket counts
// gives final positions up to the order inside a bucket, which a rank among bucket mates resolves.
__global__ void __launch_bounds__(256) k_sb_zero(Dev d) {
  const int n = d.cnt->n_start;
  for (int i = blockIdx.x * blockDim.x + threadIdx.x; i <= n; i += gridDim.x * blockDim.x) d.sb_count[i] = 0;
}

__global__ void __launch_bounds__(256) k_sb_count(Dev d) {
  const int nraw = d.cnt->n_start_raw;
  for (int i = blockIdx.x * blockDim.x + threadIdx.x; i < nraw; i += gridDim.x * blockDim.x) {
  const int h = d.start_tmp[i];
  const int sl = d.slice_of[h];
  const int m = d.slice_nstart[sl], base = d.slice_sbase[sl];
  int key = -1;
  if (base + m <= d.cnt->n_start) {  // slices beyond the capacity are dropped whole
    const float zmin = unordf(d.slice_bbox[4 * sl + 2]), zmax = unordf(d.slice_bbox[4 * sl + 3]);
    const float scale = ((float)m / fmaxf(zmax - zmin, 1e-3f)) * 0.9999f;
    int b = (int)((d.yz[h].y - zmin) * scale);
    b = max(0, min(b, m - 1));
    key = base + b;
    atomicAdd(&d.sb_count[key], 1);
  }
  d.sb_key[i] = key;
  }
}

__global__ void __launch_bounds__(256) k_sb_scatter(Dev d) {
  const int nraw = d.cnt->n_start_raw;
  for (int i = blockIdx.x * blockDim.x + threadIdx.x; i < nraw; i += gridDim.x * blockDim.x) {
    const int key = d.sb_key[i];
    if (key < 0) continue;
    const int pos = atomicAdd(&d.sb_count[key], 1);  // cursor: afterwards sb_count[key] = end of bucket key
    d.sb_sorted[pos] = d.start_tmp[i];
    d.sb_skey[pos] = key;
  }
}

__global__ void __launch_bounds__(256) k_sb_rank(Dev d) {
  const int p = blockIdx.x * blockDim.x + threadIdx.x;
  if (p >= d.cnt->n_start) return;
  const int key = d.sb_skey[p];
  const int b = key ? d.sb_count[key - 1] : 0, e = d.sb_count[key];
  const int h = d.sb_sorted[p];
  int rank = b;
  if (e - b > 1) {
    const float2 me = d.yz[h];
    const int mi = d.orig_idx[h];
    for (int q = b; q < e; q++) {
      if (q == p) continue;
      const int hq = d.sb_sorted[q];
      const float2 o = d.yz[hq];
      if (key_less(o.y, o.x, d.orig_idx[hq], me.y, me.x, mi)) rank++;
    }
  }
  d.start_hits[rank] = h;
}

void launch_clean_start(const Dev& d, Launch& L) {
  if (d.n > 0) {
    KTIMED(L, TPCCA_K_CLEAN, (k_clean<<<(d.n + 255) / 256, 256, 0, L.st>>>(d)));
    L.count++;
  }
  k_start_offsets<<<1, 1024, 0, L.st>>>(d);
  L.count++;
  if (d.n > 0 && d.max_tracklets > 0) {
    const int T = d.max_tracklets;
    k_sb_zero<<<d.n_sm * 2, 256, 0, L.st>>>(d);
    k_sb_count<<<d.n_sm * 8, 256, 0, L.st>>>(d);
    L.count += 2;
    launch_scan_i32(d.sb_count, &d.cnt->n_start, T, d.scan_tmp, L);
    k_sb_scatter<<<d.n_sm * 8, 256, 0, L.st>>>(d);
    k_sb_rank<<<(T + 255) / 256, 256, 0, L.st>>>(d);
    L.count += 2;
  }
}
