// tpcca_links.cu -- steps (b) neighbours finder, (c) neighbours cleaner, (d) start-hit finder.
// (b) PAPER.md:49 "links between hit triplets arranged close to a straight line", parallel over hits
//     (PAPER.md:57), window centred on the hit, no vertex constraint.  DESIGN.md O2.
// (c) mutual links only (north_star (c); O3).  (d) chain heads, canonical order (O4).
#include "tpcca_dev.cuh"

// ---------------------------------------------------------------- (b)
// One thread per sorted cluster; consecutive threads are neighbours in (row, y-bin, z-bin), so a warp's
// candidate ranges coincide and its loop trip counts are nearly uniform.  Two phases keep the lanes
// converged: first the down-row candidates that pass the window are collected in registers (up to
// ND_MAX), then every up-row candidate that passes is paired with them.  More than ND_MAX down
// candidates (dense noise) fall back to the plain nested loops -- same result either way.
#define ND_MAX 4

struct Best {
  int bu, bd;
  float bc;
};

__device__ __forceinline__ void consider(const Dev& d, Best& b, float cost, int u, float yu, float zu, int dd, float yd,
                                         float zd) {
  if (!(cost <= d.P.triplet_cut)) return;
  bool better;
  if (b.bu < 0) better = true;
  else if (cost != b.bc) better = cost < b.bc;
  else {  // exact tie: value-based key order (rare; keys reloaded)
    if (u != b.bu) {
      const float2 q = d.yz[b.bu];
      better = key_less(zu, yu, d.orig_idx[u], q.y, q.x, d.orig_idx[b.bu]);
    } else {
      const float2 q = d.yz[b.bd];
      better = key_less(zd, yd, d.orig_idx[dd], q.y, q.x, d.orig_idx[b.bd]);
    }
  }
  if (better) { b.bu = u; b.bd = dd; b.bc = cost; }
}

__global__ void __launch_bounds__(128) k_neighbours(Dev d) {
  const int h = blockIdx.x * blockDim.x + threadIdx.x;
  if (h >= d.n) return;
  const int sl = d.slice_of[h];
  const NbrHdr nb = d.nbr[sl];
  Best best;
  best.bu = -1; best.bd = -1; best.bc = 0.0f;
  if (nb.su >= 0) {
    const float2 p0 = d.yz[h];
    const float y0 = p0.x, z0 = p0.y;
    const float t = nb.t;
    const float mz = 1e-3f + fabsf(z0) * 4e-7f;
    const GridHdr gu = d.grid[nb.su];
    const GridHdr gd = d.grid[nb.sd];
    int uy0, uy1, uz0, uz1, dy0, dy1, dz0, dz1;
    bin_range(y0 - nb.wyu - 1e-3f, y0 + nb.wyu + 1e-3f, gu.ymin, gu.inv_by, gu.ny, uy0, uy1);
    bin_range(z0 - nb.wzu - mz, z0 + nb.wzu + mz, gu.zmin, gu.inv_bz, gu.nz, uz0, uz1);
    bin_range(y0 - nb.wyd - 1e-3f, y0 + nb.wyd + 1e-3f, gd.ymin, gd.inv_by, gd.ny, dy0, dy1);
    bin_range(z0 - nb.wzd - mz, z0 + nb.wzd + mz, gd.zmin, gd.inv_bz, gd.nz, dz0, dz1);
    if (uz0 <= uz1 && dz0 <= dz1) {
      // phase 1: down-row candidates inside the window
      float cy[ND_MAX], cz[ND_MAX];
      int ci[ND_MAX];
      int nd = 0;
      for (int by = dy0; by <= dy1; by++) {
        const int* bs = d.bin_start + gd.bin_base + by * gd.nz;
        const int cb = bs[dz0], ce = bs[dz1 + 1];
        for (int c = cb; c < ce; c++) {
          const float2 p = d.yz[c];
          if (!(fabsf(p.x - y0) <= nb.wyd) || !(fabsf(p.y - z0) <= nb.wzd)) continue;
#pragma unroll
          for (int j = 0; j < ND_MAX; j++)
            if (j == nd) { cy[j] = p.x; cz[j] = p.y; ci[j] = c; }
          nd++;
        }
      }
      if (nd > 0) {
        // phase 2: up-row candidates, paired with the collected down candidates
        for (int by = uy0; by <= uy1; by++) {
          const int* bs = d.bin_start + gu.bin_base + by * gu.nz;
          const int ub = bs[uz0], ue = bs[uz1 + 1];
          for (int u = ub; u < ue; u++) {
            const float2 pu = d.yz[u];
            if (!(fabsf(pu.x - y0) <= nb.wyu) || !(fabsf(pu.y - z0) <= nb.wzu)) continue;
            if (nd <= ND_MAX) {
#pragma unroll
              for (int j = 0; j < ND_MAX; j++) {
                if (j < nd) {
                  const float ey = y0 - (cy[j] + t * (pu.x - cy[j]));
                  const float ez = z0 - (cz[j] + t * (pu.y - cz[j]));
                  const float cost = (ey * ey) * d.inv_sy2 + (ez * ez) * d.inv_sz2;
                  consider(d, best, cost, u, pu.x, pu.y, ci[j], cy[j], cz[j]);
                }
              }
            } else {  // overflow: plain nested loop over the down row
              for (int by2 = dy0; by2 <= dy1; by2++) {
                const int* bs2 = d.bin_start + gd.bin_base + by2 * gd.nz;
                const int db = bs2[dz0], de = bs2[dz1 + 1];
                for (int dd = db; dd < de; dd++) {
                  const float2 pd = d.yz[dd];
                  if (!(fabsf(pd.x - y0) <= nb.wyd) || !(fabsf(pd.y - z0) <= nb.wzd)) continue;
                  const float ey = y0 - (pd.x + t * (pu.x - pd.x));
                  const float ez = z0 - (pd.y + t * (pu.y - pd.y));
                  const float cost = (ey * ey) * d.inv_sy2 + (ez * ez) * d.inv_sz2;
                  consider(d, best, cost, u, pu.x, pu.y, dd, pd.x, pd.y);
                }
              }
            }
          }
        }
      }
    }
  }
  d.link_up[h] = best.bu;
  d.link_down[h] = best.bd;
}

void launch_neighbours(const Dev& d, Launch& L) {
  if (d.n <= 0) return;
  k_neighbours<<<(d.n + 127) / 128, 128, 0, L.st>>>(d);
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
  if (h < d.n) {
    int u = d.link_up[h], dn = d.link_down[h];
    if (u >= 0 && d.link_down[u] != h) u = -1;
    if (dn >= 0 && d.link_up[dn] != h) dn = -1;
    d.link_up_clean[h] = u;
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
    k_clean<<<(d.n + 255) / 256, 256, 0, L.st>>>(d);
    L.count++;
  }
  k_start_offsets<<<1, 1024, 0, L.st>>>(d);
  L.count++;
  if (d.n > 0 && d.max_tracklets > 0) {
    const int T = d.max_tracklets;
    k_sb_zero<<<148 * 2, 256, 0, L.st>>>(d);
    k_sb_count<<<148 * 8, 256, 0, L.st>>>(d);
    L.count += 2;
    launch_scan_i32(d.sb_count, &d.cnt->n_start, T, d.scan_tmp, L);
    k_sb_scatter<<<148 * 8, 256, 0, L.st>>>(d);
    k_sb_rank<<<(T + 255) / 256, 256, 0, L.st>>>(d);
    L.count += 2;
  }
}
