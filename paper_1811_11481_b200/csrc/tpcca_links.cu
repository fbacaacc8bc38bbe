// tpcca_links.cu -- steps (b) neighbours finder, (c) neighbours cleaner, (d) start-hit finder.
// (b) PAPER.md:49 "links between hit triplets arranged close to a straight line", parallel over hits
//     (PAPER.md:57), window centred on the hit, no vertex constraint.  DESIGN.md O2.
// (c) mutual links only (north_star (c); O3).  (d) chain heads, canonical order (O4).
#include "tpcca_dev.cuh"

// ---------------------------------------------------------------- (b)
// One thread per sorted cluster.  Consecutive threads are neighbours in (row, y-bin, z-bin), so their
// candidate ranges overlap in L1.
struct RowWin {
  int sl;          // slice of the neighbour row, -1 none
  float wy, wz;    // window half widths (exact predicate)
};

__device__ __forceinline__ int pick_row(const Dev& d, int sec, int r, int dir) {
  const int r1 = r + dir, r2 = r + 2 * dir;
  if (r1 >= 0 && r1 < d.n_rows) {
    const int sl = sec * d.n_rows + r1;
    if (d.row_start[sl + 1] > d.row_start[sl]) return r1;
  }
  if (r2 >= 0 && r2 < d.n_rows) {
    const int sl = sec * d.n_rows + r2;
    if (d.row_start[sl + 1] > d.row_start[sl]) return r2;
  }
  return -1;
}

__global__ void __launch_bounds__(128) k_neighbours(Dev d) {
  const int h = blockIdx.x * blockDim.x + threadIdx.x;
  if (h >= d.n) return;
  const int sl = d.slice_of[h];
  const int sec = sl / d.n_rows, r = sl - sec * d.n_rows;
  const int ru = pick_row(d, sec, r, +1), rd = pick_row(d, sec, r, -1);
  int bu = -1, bd = -1;
  if (ru >= 0 && rd >= 0) {
    const float xr = d.row_x[r];
    const float dxu = d.row_x[ru] - xr;
    const float dxd = xr - d.row_x[rd];
    const float t = dxd / (dxu + dxd);
    const float wyu = dxu * d.P.nbr_dydx + d.P.nbr_margin_y;
    const float wzu = dxu * d.P.nbr_dzdx + d.P.nbr_margin_z;
    const float wyd = dxd * d.P.nbr_dydx + d.P.nbr_margin_y;
    const float wzd = dxd * d.P.nbr_dzdx + d.P.nbr_margin_z;
    const float2 p0 = d.yz[h];
    const float y0 = p0.x, z0 = p0.y;
    const float mz = 1e-3f + fabsf(z0) * 4e-7f;
    const GridHdr gu = d.grid[sec * d.n_rows + ru];
    const GridHdr gd = d.grid[sec * d.n_rows + rd];
    int uy0, uy1, uz0, uz1, dy0, dy1, dz0, dz1;
    bin_range(y0 - wyu - 1e-3f, y0 + wyu + 1e-3f, gu.ymin, gu.inv_by, gu.ny, uy0, uy1);
    bin_range(z0 - wzu - mz, z0 + wzu + mz, gu.zmin, gu.inv_bz, gu.nz, uz0, uz1);
    bin_range(y0 - wyd - 1e-3f, y0 + wyd + 1e-3f, gd.ymin, gd.inv_by, gd.ny, dy0, dy1);
    bin_range(z0 - wzd - mz, z0 + wzd + mz, gd.zmin, gd.inv_bz, gd.nz, dz0, dz1);
    float bc = 0.0f, buy = 0.0f, buz = 0.0f, bdy = 0.0f, bdz = 0.0f;
    if (uz0 <= uz1 && dz0 <= dz1) {
      for (int uy = uy0; uy <= uy1; uy++) {
        const int ub = d.bin_start[gu.bin_base + uy * gu.nz + uz0];
        const int ue = d.bin_start[gu.bin_base + uy * gu.nz + uz1 + 1];
        for (int u = ub; u < ue; u++) {
          const float2 pu = d.yz[u];
          if (!(fabsf(pu.x - y0) <= wyu) || !(fabsf(pu.y - z0) <= wzu)) continue;
          for (int dy = dy0; dy <= dy1; dy++) {
            const int db = d.bin_start[gd.bin_base + dy * gd.nz + dz0];
            const int de = d.bin_start[gd.bin_base + dy * gd.nz + dz1 + 1];
            for (int dd = db; dd < de; dd++) {
              const float2 pd = d.yz[dd];
              if (!(fabsf(pd.x - y0) <= wyd) || !(fabsf(pd.y - z0) <= wzd)) continue;
              const float ey = y0 - (pd.x + t * (pu.x - pd.x));
              const float ez = z0 - (pd.y + t * (pu.y - pd.y));
              const float cost = (ey * ey) * d.inv_sy2 + (ez * ez) * d.inv_sz2;
              if (!(cost <= d.P.triplet_cut)) continue;
              bool better;
              if (bu < 0) better = true;
              else if (cost != bc) better = cost < bc;
              else if (u != bu) better = key_less(pu.y, pu.x, d.orig_idx[u], buz, buy, d.orig_idx[bu]);
              else better = key_less(pd.y, pd.x, d.orig_idx[dd], bdz, bdy, d.orig_idx[bd]);
              if (better) { bu = u; bd = dd; bc = cost; buy = pu.x; buz = pu.y; bdy = pd.x; bdz = pd.y; }
            }
          }
        }
      }
    }
  }
  d.link_up[h] = bu;
  d.link_down[h] = bd;
}

void launch_neighbours(const Dev& d, Launch& L) {
  if (d.n <= 0) return;
  k_neighbours<<<(d.n + 127) / 128, 128, 0, L.st>>>(d);
  L.count++;
}

// ---------------------------------------------------------------- (c) + (d1)
__global__ void __launch_bounds__(256) k_clean(Dev d) {
  const int h = blockIdx.x * blockDim.x + threadIdx.x;
  if (h >= d.n) return;
  int u = d.link_up[h], dn = d.link_down[h];
  if (u >= 0 && d.link_down[u] != h) u = -1;
  if (dn >= 0 && d.link_up[dn] != h) dn = -1;
  d.link_up_clean[h] = u;
  const bool start = (dn < 0) && (u >= 0);
  d.start_flag[h] = start ? 1 : 0;
  if (start) atomicAdd(&d.slice_nstart[d.slice_of[h]], 1);
}

// (d2) exclusive scan of per-slice start counts
__global__ void __launch_bounds__(1024) k_start_offsets(Dev d) {
  __shared__ int sm[32];
  int carry = 0;
  for (int b0 = 0; b0 < d.n_slices; b0 += 1024) {
    const int sl = b0 + threadIdx.x;
    const int v = (sl < d.n_slices) ? d.slice_nstart[sl] : 0;
    int tot;
    const int e = block_scan_excl(v, &tot, sm);
    if (sl < d.n_slices) d.slice_sbase[sl] = carry + e;
    carry += tot;
  }
  if (threadIdx.x == 0) {
    d.slice_sbase[d.n_slices] = carry;
    if (carry > d.max_tracklets) atomicOr(&d.cnt->status, TPCCA_STAT_TRACKLET_OVERFLOW);
    d.cnt->n_start = min(carry, d.max_tracklets);
  }
}

// (d3) one block per slice: gather its start hits, rank-sort them by key (ord z, ord y, input index)
#define D3_THREADS 128
__global__ void __launch_bounds__(D3_THREADS) k_start_sort(Dev d) {
  const int sl = blockIdx.x;
  const int m = d.slice_nstart[sl];
  if (m == 0) return;
  const int sbase = d.slice_sbase[sl];
  if (sbase >= d.max_tracklets) return;
  const int mm = min(m, d.max_tracklets - sbase);  // overflow: deterministic only when not truncated
  __shared__ int s_n;
  __shared__ float s_z[D3_THREADS], s_y[D3_THREADS];
  __shared__ int s_i[D3_THREADS];
  if (threadIdx.x == 0) s_n = 0;
  __syncthreads();
  const int b = d.row_start[sl], e = d.row_start[sl + 1];
  for (int h = b + threadIdx.x; h < e; h += D3_THREADS)
    if (d.start_flag[h]) {
      const int k = atomicAdd(&s_n, 1);
      if (k < mm) d.start_tmp[sbase + k] = h;
    }
  __syncthreads();
  for (int i0 = 0; i0 < mm; i0 += D3_THREADS) {
    const int i = i0 + threadIdx.x;
    int hi = -1, ii = 0, rank = 0;
    float zi = 0.0f, yi = 0.0f;
    if (i < mm) {
      hi = d.start_tmp[sbase + i];
      const float2 p = d.yz[hi];
      yi = p.x; zi = p.y; ii = d.orig_idx[hi];
    }
    for (int j0 = 0; j0 < mm; j0 += D3_THREADS) {
      __syncthreads();
      const int j = j0 + threadIdx.x;
      if (j < mm) {
        const int hj = d.start_tmp[sbase + j];
        const float2 p = d.yz[hj];
        s_y[threadIdx.x] = p.x; s_z[threadIdx.x] = p.y; s_i[threadIdx.x] = d.orig_idx[hj];
      }
      __syncthreads();
      const int cntj = min(D3_THREADS, mm - j0);
      if (i < mm)
        for (int j2 = 0; j2 < cntj; j2++)
          if (key_less(s_z[j2], s_y[j2], s_i[j2], zi, yi, ii)) rank++;
    }
    if (i < mm) d.start_hits[sbase + rank] = hi;
  }
}

void launch_clean_start(const Dev& d, Launch& L) {
  if (d.n > 0) {
    k_clean<<<(d.n + 255) / 256, 256, 0, L.st>>>(d);
    L.count++;
  }
  k_start_offsets<<<1, 1024, 0, L.st>>>(d);
  L.count++;
  if (d.n > 0) {
    k_start_sort<<<d.n_slices, D3_THREADS, 0, L.st>>>(d);
    L.count++;
  }
}
