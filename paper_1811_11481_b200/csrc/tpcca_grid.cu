// tpcca_grid.cu -- step (a): cluster grid builder (north_star (a); PAPER.md:49 sectors, :41 pad rows).
// Counting sort of the frame's clusters by (sector, row) slice and, inside a slice, by a 2-D (y,z) bin
// grid: histogram -> exclusive scan -> scatter.  The grid is an acceleration structure only (DESIGN.md
// O1/A3): no tracking result depends on bin sizes or on the order of clusters inside a bin.
#include "tpcca_dev.cuh"

// ---------------------------------------------------------------- generic exclusive scan (int32)
#define SCAN_THREADS 512
#define SCAN_ITEMS 4
#define SCAN_TILE (SCAN_THREADS * SCAN_ITEMS)

__global__ void __launch_bounds__(SCAN_THREADS) k_scan_reduce(const int32_t* __restrict__ data,
                                                              const int32_t* __restrict__ n_dev, int32_t n_max,
                                                              int32_t* __restrict__ partial) {
  __shared__ int sm[32];
  const int n = min(*n_dev, n_max);
  const int base = blockIdx.x * SCAN_TILE;
  if (base >= n) return;
  int v = 0;
#pragma unroll
  for (int k = 0; k < SCAN_ITEMS; k++) {
    const int i = base + k * SCAN_THREADS + threadIdx.x;
    if (i < n) v += data[i];
  }
  int tot;
  block_scan_excl(v, &tot, sm);
  if (threadIdx.x == 0) partial[blockIdx.x] = tot;
}

__global__ void __launch_bounds__(1024) k_scan_partials(int32_t* __restrict__ partial,
                                                        const int32_t* __restrict__ n_dev, int32_t n_max) {
  __shared__ int sm[32];
  const int n = min(*n_dev, n_max);
  const int nb = (n + SCAN_TILE - 1) / SCAN_TILE;
  int carry = 0;
  for (int b0 = 0; b0 < nb; b0 += 1024) {
    const int i = b0 + threadIdx.x;
    const int v = (i < nb) ? partial[i] : 0;
    int tot;
    const int e = block_scan_excl(v, &tot, sm);
    if (i < nb) partial[i] = carry + e;
    carry += tot;
  }
  if (threadIdx.x == 0) partial[nb] = carry;
}

__global__ void __launch_bounds__(SCAN_THREADS) k_scan_down(int32_t* __restrict__ data,
                                                            const int32_t* __restrict__ n_dev, int32_t n_max,
                                                            const int32_t* __restrict__ partial) {
  __shared__ int sm[32];
  const int n = min(*n_dev, n_max);
  const int base = blockIdx.x * SCAN_TILE;
  if (base >= n) return;
  // blocked arrangement: thread t owns items [t*ITEMS, t*ITEMS+ITEMS)
  int v[SCAN_ITEMS], s = 0;
#pragma unroll
  for (int k = 0; k < SCAN_ITEMS; k++) {
    const int i = base + threadIdx.x * SCAN_ITEMS + k;
    v[k] = (i < n) ? data[i] : 0;
    s += v[k];
  }
  int tot;
  int e = block_scan_excl(s, &tot, sm) + partial[blockIdx.x];
#pragma unroll
  for (int k = 0; k < SCAN_ITEMS; k++) {
    const int i = base + threadIdx.x * SCAN_ITEMS + k;
    if (i < n) data[i] = e;
    e += v[k];
  }
  const int nb = (n + SCAN_TILE - 1) / SCAN_TILE;
  if (blockIdx.x == nb - 1 && threadIdx.x == 0) data[n] = partial[nb];
}

__global__ void k_scan_empty(int32_t* data, const int32_t* n_dev) {
  if (*n_dev <= 0) data[0] = 0;
}

void launch_scan_i32(int32_t* data, const int32_t* n_dev, int32_t n_max, int32_t* tmp, Launch& L) {
  const int nb = (n_max + SCAN_TILE - 1) / SCAN_TILE;
  if (nb == 0) { k_scan_empty<<<1, 1, 0, L.st>>>(data, n_dev); L.count++; return; }
  k_scan_reduce<<<nb, SCAN_THREADS, 0, L.st>>>(data, n_dev, n_max, tmp);
  k_scan_partials<<<1, 1024, 0, L.st>>>(tmp, n_dev, n_max);
  k_scan_down<<<nb, SCAN_THREADS, 0, L.st>>>(data, n_dev, n_max, tmp);
  k_scan_empty<<<1, 1, 0, L.st>>>(data, n_dev);
  L.count += 4;
}

// ---------------------------------------------------------------- counting sort by decreasing key (work orders)
// Longest-first work orders for the persistent Kalman kernels and the refit: lanes of a warp then run about the
// same number of row steps and the short items fill the tail.  ord = [hist 0..511 | cursors 512..1023], zeroed.
#define ORD_THREADS 1024
#define ORD_KEYS 257
__global__ void __launch_bounds__(ORD_THREADS) k_order_hist(int32_t* __restrict__ ord, const int32_t* __restrict__ key,
                                                            const int32_t* __restrict__ n_dev, int32_t n_max) {
  __shared__ int s_hist[ORD_KEYS];
  const int n = min(*n_dev, n_max);
  if (blockIdx.x * ORD_THREADS >= n) return;
  for (int i = threadIdx.x; i < ORD_KEYS; i += ORD_THREADS) s_hist[i] = 0;
  __syncthreads();
  const int i = blockIdx.x * ORD_THREADS + threadIdx.x;
  if (i < n) atomicAdd(&s_hist[min(max(key[i], 0), ORD_KEYS - 1)], 1);
  __syncthreads();
  for (int k = threadIdx.x; k < ORD_KEYS; k += ORD_THREADS)
    if (s_hist[k]) atomicAdd(&ord[k], s_hist[k]);
}
__global__ void __launch_bounds__(512) k_order_offsets(int32_t* __restrict__ ord) {
  __shared__ int sm[32];
  const int i = threadIdx.x;  // position i holds key ORD_KEYS-1-i
  const int v = (i < ORD_KEYS) ? ord[ORD_KEYS - 1 - i] : 0;
  int tot;
  const int e = block_scan_excl(v, &tot, sm);
  if (i < ORD_KEYS) ord[512 + ORD_KEYS - 1 - i] = e;
}
__global__ void __launch_bounds__(ORD_THREADS) k_order_scatter(int32_t* __restrict__ ord, const int32_t* __restrict__ key,
                                                               const int32_t* __restrict__ n_dev, int32_t n_max,
                                                               int32_t* __restrict__ out) {
  __shared__ int s_cnt[ORD_KEYS], s_base[ORD_KEYS];
  const int n = min(*n_dev, n_max);
  if (blockIdx.x * ORD_THREADS >= n) return;
  for (int i = threadIdx.x; i < ORD_KEYS; i += ORD_THREADS) s_cnt[i] = 0;
  __syncthreads();
  const int i = blockIdx.x * ORD_THREADS + threadIdx.x;
  int k = 0, rank = 0;
  if (i < n) {
    k = min(max(key[i], 0), ORD_KEYS - 1);
    rank = atomicAdd(&s_cnt[k], 1);
  }
  __syncthreads();
  for (int q = threadIdx.x; q < ORD_KEYS; q += ORD_THREADS)
    if (s_cnt[q]) s_base[q] = atomicAdd(&ord[512 + q], s_cnt[q]);
  __syncthreads();
  if (i < n) out[s_base[k] + rank] = i;
}

void launch_order_desc(const Dev& d, int slot, const int32_t* key, const int32_t* n_dev, int32_t n_max, int32_t* out,
                       Launch& L) {
  if (n_max <= 0) return;
  int32_t* ord = d.ord + 1024 * slot;
  const int nb = (n_max + ORD_THREADS - 1) / ORD_THREADS;
  k_order_hist<<<nb, ORD_THREADS, 0, L.st>>>(ord, key, n_dev, n_max);
  k_order_offsets<<<1, 512, 0, L.st>>>(ord);
  k_order_scatter<<<nb, ORD_THREADS, 0, L.st>>>(ord, key, n_dev, n_max, out);
  L.count += 3;
}

// ---------------------------------------------------------------- (a0) reset per-call state
__global__ void k_reset(Dev d) {
  const int i = blockIdx.x * blockDim.x + threadIdx.x;
  if (i <= d.n_slices) {
    d.slice_count[i] = 0;
    d.slice_nstart[i] = 0;
  }
  if (i < d.n_slices) {
    d.slice_bbox[4 * i + 0] = 0xFFFFFFFFu;  // ymin
    d.slice_bbox[4 * i + 1] = 0u;           // ymax
    d.slice_bbox[4 * i + 2] = 0xFFFFFFFFu;  // zmin
    d.slice_bbox[4 * i + 3] = 0u;           // zmax
  }
  if (i < 4 * 1024) d.ord[i] = 0;
  if (i == 0) {
    d.cnt->n_start = 0; d.cnt->n_tracks = 0; d.cnt->n_valid = 0; d.cnt->status = 0; d.cnt->n_bins = 0; d.cnt->n_start_raw = 0; d.cnt->n_work = 0; d.cnt->work_next[0] = 0; d.cnt->work_next[1] = 0; d.cnt->work_next[2] = 0; d.cnt->work_next[3] = 0;
    d.cnt->row_steps = 0ull; d.cnt->searches = 0ull; d.cnt->track_hits = 0ull;
  }
}

// ---------------------------------------------------------------- (a1) slice histogram + bounding boxes
#define A1_THREADS 256
#define A1_ITEMS 8
__global__ void __launch_bounds__(A1_THREADS) k_slice_count(Dev d, SecOff so) {
  __shared__ int s_cnt[TPCCA_MAX_ROWS];
  __shared__ uint32_t s_box[TPCCA_MAX_ROWS * 4];
  const int base = blockIdx.x * (A1_THREADS * A1_ITEMS);
  const int sec0 = sector_of(so, d.n_sectors, min(base, d.n - 1));  // sector privatised in shared memory
  for (int r = threadIdx.x; r < d.n_rows; r += A1_THREADS) {
    s_cnt[r] = 0;
    s_box[4 * r] = 0xFFFFFFFFu; s_box[4 * r + 1] = 0u; s_box[4 * r + 2] = 0xFFFFFFFFu; s_box[4 * r + 3] = 0u;
  }
  __syncthreads();
  bool bad = false;
#pragma unroll
  for (int k = 0; k < A1_ITEMS; k++) {
    const int i = base + k * A1_THREADS + threadIdx.x;
    if (i >= d.n) continue;
    const float4 c = __ldg(&d.clusters[i]);
    const int row = __float_as_int(c.w);
    if (row < 0 || row >= d.n_rows) { bad = true; continue; }
    const int sec = (i < so.v[sec0 + 1]) ? sec0 : sector_of(so, d.n_sectors, i);
    const uint32_t oy = ordf(c.y), oz = ordf(c.z);
    if (sec == sec0) {
      atomicAdd(&s_cnt[row], 1);
      atomicMin(&s_box[4 * row], oy); atomicMax(&s_box[4 * row + 1], oy);
      atomicMin(&s_box[4 * row + 2], oz); atomicMax(&s_box[4 * row + 3], oz);
    } else {
      const int sl = sec * d.n_rows + row;
      atomicAdd(&d.slice_count[sl], 1);
      atomicMin(&d.slice_bbox[4 * sl], oy); atomicMax(&d.slice_bbox[4 * sl + 1], oy);
      atomicMin(&d.slice_bbox[4 * sl + 2], oz); atomicMax(&d.slice_bbox[4 * sl + 3], oz);
    }
  }
  if (bad) atomicOr(&d.cnt->status, TPCCA_STAT_BAD_CLUSTER);
  __syncthreads();
  for (int r = threadIdx.x; r < d.n_rows; r += A1_THREADS) {
    const int c = s_cnt[r];
    if (c) {
      const int sl = sec0 * d.n_rows + r;
      atomicAdd(&d.slice_count[sl], c);
      atomicMin(&d.slice_bbox[4 * sl], s_box[4 * r]); atomicMax(&d.slice_bbox[4 * sl + 1], s_box[4 * r + 1]);
      atomicMin(&d.slice_bbox[4 * sl + 2], s_box[4 * r + 2]); atomicMax(&d.slice_bbox[4 * sl + 3], s_box[4 * r + 3]);
    }
  }
}

// ---------------------------------------------------------------- (a2) slice offsets + grid headers
__global__ void __launch_bounds__(1024) k_slice_setup(Dev d) {
  __shared__ int sm[32];
  int carry_c = 0, carry_b = 0;
  for (int b0 = 0; b0 < d.n_slices; b0 += 1024) {
    const int sl = b0 + threadIdx.x;
    int cnt = 0, nb = 0;
    GridHdr g;
    g.ymin = g.zmin = 0.0f; g.inv_by = g.inv_bz = 0.0f; g.ny = g.nz = 1; g.bin_base = 0; g.pad = 0;
    if (sl < d.n_slices) {
      cnt = d.slice_count[sl];
      if (cnt > 0) {
        const float ymin = unordf(d.slice_bbox[4 * sl]), ymax = unordf(d.slice_bbox[4 * sl + 1]);
        const float zmin = unordf(d.slice_bbox[4 * sl + 2]), zmax = unordf(d.slice_bbox[4 * sl + 3]);
        const float ye = fmaxf(ymax - ymin, 1e-3f), ze = fmaxf(zmax - zmin, 1e-3f);
        int ny = (int)(ye / d.P.grid_bin_y) + 1;
        ny = min(ny, 128);
        float want = (float)cnt * d.P.grid_bins_per_cluster / (float)ny;
        int nz = (int)want + 1;
        const int nz_cap = (int)fminf(ze / d.P.grid_bin_z_min, 1.0e6f) + 1;
        nz = max(1, min(nz, nz_cap));
        g.ymin = ymin; g.zmin = zmin;
        g.inv_by = ((float)ny / ye) * 0.9999f;
        g.inv_bz = ((float)nz / ze) * 0.9999f;
        g.ny = ny; g.nz = nz; g.pad = cnt;
        nb = ny * nz;
      }
    }
    int tot_c, tot_b;
    const int ec = block_scan_excl(cnt, &tot_c, sm);
    const int eb = block_scan_excl(nb, &tot_b, sm);
    if (sl < d.n_slices) {
      d.row_start[sl] = carry_c + ec;
      g.bin_base = carry_b + eb;
      if (g.bin_base + nb > d.max_bins) {  // cannot happen with the default sizing; degrade to one bin
        g.ny = g.nz = 1; g.pad = 0; g.bin_base = min(g.bin_base, d.max_bins - 1);
        atomicOr(&d.cnt->status, TPCCA_STAT_BIN_OVERFLOW);
      }
      d.grid[sl] = g;
      // per-row constants of the neighbours finder (O2): up/down row with one skip
      const int sec = sl / d.n_rows, r = sl - sec * d.n_rows;
      NbrHdr nb;
      nb.su = nb.sd = -1; nb.t = nb.wyu = nb.wzu = nb.wyd = nb.wzd = 0.0f; nb.pad = 0;
      int ru = -1, rd = -1;
      if (r + 1 < d.n_rows && d.slice_count[sl + 1] > 0) ru = r + 1;
      else if (r + 2 < d.n_rows && d.slice_count[sl + 2] > 0) ru = r + 2;
      if (r - 1 >= 0 && d.slice_count[sl - 1] > 0) rd = r - 1;
      else if (r - 2 >= 0 && d.slice_count[sl - 2] > 0) rd = r - 2;
      if (ru >= 0 && rd >= 0 && cnt > 0) {
        const float xr = d.row_x[r];
        const float dxu = d.row_x[ru] - xr;
        const float dxd = xr - d.row_x[rd];
        nb.su = sec * d.n_rows + ru; nb.sd = sec * d.n_rows + rd;
        nb.t = dxd / (dxu + dxd);
        nb.wyu = dxu * d.P.nbr_dydx + d.P.nbr_margin_y;
        nb.wzu = dxu * d.P.nbr_dzdx + d.P.nbr_margin_z;
        nb.wyd = dxd * d.P.nbr_dydx + d.P.nbr_margin_y;
        nb.wzd = dxd * d.P.nbr_dzdx + d.P.nbr_margin_z;
      }
      d.nbr[sl] = nb;
    }
    carry_c += tot_c;
    carry_b += tot_b;
  }
  if (threadIdx.x == 0) {
    d.row_start[d.n_slices] = carry_c;
    d.cnt->n_bins = min(carry_b, d.max_bins);
  }
}

__global__ void k_zero_bins(Dev d) {
  const int n = d.cnt->n_bins;
  for (int i = blockIdx.x * blockDim.x + threadIdx.x; i <= n; i += gridDim.x * blockDim.x) d.bin_start[i] = 0;
  // hit weights of the selector: cleared here with coalesced stores rather than in the scatter
  ulonglong2* hw = reinterpret_cast<ulonglong2*>(d.hit_weight);
  const int n2 = (d.n + 1) >> 1;  // the array is 256-byte aligned and padded
  for (int i = blockIdx.x * blockDim.x + threadIdx.x; i < n2; i += gridDim.x * blockDim.x) hw[i] = make_ulonglong2(0ull, 0ull);
}

// ---------------------------------------------------------------- (a3) bin histogram (rank = arrival order)
__global__ void __launch_bounds__(256) k_bin_count(Dev d, SecOff so) {
  const int i = blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= d.n) return;
  const float4 c = __ldg(&d.clusters[i]);
  const int row = __float_as_int(c.w);
  if (row < 0 || row >= d.n_rows) { d.cluster_bin[i] = -1; return; }
  const int sl = sector_of(so, d.n_sectors, i) * d.n_rows + row;
  const GridHdr g = d.grid[sl];
  int by = (int)((c.y - g.ymin) * g.inv_by);
  int bz = (int)((c.z - g.zmin) * g.inv_bz);
  by = max(0, min(by, g.ny - 1));
  bz = max(0, min(bz, g.nz - 1));
  const int gb = g.bin_base + by * g.nz + bz;
  d.cluster_bin[i] = gb;
  d.cluster_rank[i] = atomicAdd(&d.bin_start[gb], 1);
}

// ---------------------------------------------------------------- (a4) scatter into sorted SoA
__global__ void __launch_bounds__(256) k_scatter(Dev d, SecOff so) {
  const int i = blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= d.n) return;
  const int gb = d.cluster_bin[i];
  if (gb < 0) { d.out_assign[i] = -1; return; }
  const float4 c = __ldg(&d.clusters[i]);
  const int pos = d.bin_start[gb] + d.cluster_rank[i];
  d.yz[pos] = make_float2(c.y, c.z);
  d.orig_idx[pos] = i;
}

// slice id of every sorted position: one block per slice, coalesced stores (instead of a 2-byte scatter)
__global__ void __launch_bounds__(128) k_fill_slice_of(Dev d) {
  const int sl = blockIdx.x;
  const int b = d.row_start[sl], e = d.row_start[sl + 1];
  for (int i = b + threadIdx.x; i < e; i += blockDim.x) d.slice_of[i] = (uint16_t)sl;
}

void launch_grid(const Dev& d, const SecOff& so, Launch& L) {
  k_reset<<<(max(d.n_slices, 4 * 1024) + 256) / 256, 256, 0, L.st>>>(d);
  L.count++;
  if (d.n > 0) {
    k_slice_count<<<(d.n + A1_THREADS * A1_ITEMS - 1) / (A1_THREADS * A1_ITEMS), A1_THREADS, 0, L.st>>>(d, so);
    L.count++;
  }
  k_slice_setup<<<1, 1024, 0, L.st>>>(d);
  k_zero_bins<<<148 * 4, 256, 0, L.st>>>(d);
  L.count += 2;
  if (d.n > 0) {
    k_bin_count<<<(d.n + 255) / 256, 256, 0, L.st>>>(d, so);
    L.count++;
    launch_scan_i32(d.bin_start, &d.cnt->n_bins, d.max_bins, d.scan_tmp, L);
    k_scatter<<<(d.n + 255) / 256, 256, 0, L.st>>>(d, so);
    k_fill_slice_of<<<d.n_slices, 128, 0, L.st>>>(d);
    L.count += 2;
  }
}
