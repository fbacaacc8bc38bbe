// tpcca_grid.cu -- step (a): cluster grid builder (north_star (a); PAPER.md:49 sectors, :41 pad rows).
// Counting sort of the frame's clusters by (sector, row) slice and, inside a slice, by a 2-D (y,z) bin
// grid: histogram -> exclusive scan -> scatter, in two levels (slices, then bins inside a slice).  The grid is an acceleration structure only (DESIGN.md
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
#define ORD_SLOTS 5  // counting-sort scratch blocks of Dev::ord (refit, E2, E3a, E3b, merged fit)
__global__ void k_reset(Dev d) {
  const int stride = gridDim.x * blockDim.x;
  for (int i = blockIdx.x * blockDim.x + threadIdx.x; i <= d.n_slices; i += stride) {
    d.slice_count[i] = 0;
    d.slice_nstart[i] = 0;
    if (i < d.n_slices) {
      d.slice_bbox[4 * i + 0] = 0xFFFFFFFFu;  // ymin
      d.slice_bbox[4 * i + 1] = 0u;           // ymax
      d.slice_bbox[4 * i + 2] = 0xFFFFFFFFu;  // zmin
      d.slice_bbox[4 * i + 3] = 0u;           // zmax
    }
  }
  for (int i = blockIdx.x * blockDim.x + threadIdx.x; i < ORD_SLOTS * 1024; i += stride) d.ord[i] = 0;
  if (blockIdx.x == 0 && threadIdx.x == 0) {
    d.cnt->n_start = 0; d.cnt->n_tracks = 0; d.cnt->n_valid = 0; d.cnt->status = 0; d.cnt->n_bins = 0;
    d.cnt->n_start_raw = 0; d.cnt->n_work = 0;
    d.cnt->n_merged = 0; d.cnt->n_links = 0; d.cnt->n_fit_failed = 0; d.cnt->pad0 = 0;
    for (int q = 0; q < 4; q++) d.cnt->work_next[q] = 0;
    d.cnt->row_steps = 0ull; d.cnt->searches = 0ull; d.cnt->track_hits = 0ull; d.cnt->tracklet_hits = 0ull;
    for (int q = 0; q < 4; q++) d.cnt->phase_steps[q] = 0ull;
  }
}

// ---------------------------------------------------------------- (a) grid builder, two levels
// Level 1 moves the clusters into (sector, row) slice order as 16-byte records: a slice histogram, one small scan,
// then a scatter in which every block reserves its rows' ranges once (block-local ranks in shared memory), so that a
// block's clusters of one row land next to each other.  Level 2 runs one block per slice on the slice's contiguous
// records (L1/L2 resident): bounding box, grid header, bin histogram and cursors in shared memory, and the final
// (y-bin, z-bin) order written to yz / orig_idx / slice_of together with the slice's piece of bin_start.
// Bins are laid out by an upper bound that depends on the slice counts alone (bins_per_cluster * count + 129 per
// slice), so the grid dimensions -- which need the bounding box -- can be chosen inside level 2.
#define A1_THREADS 256
#define A1_ITEMS 8
#define A1_TILE (A1_THREADS * A1_ITEMS)

// a cluster with a non-finite y or z is ignored like one with a bad row (A21)
__device__ __forceinline__ bool cluster_finite(const float4& c) {
  return fabsf(c.y) <= 3.0e38f && fabsf(c.z) <= 3.0e38f;  // false for NaN and +-inf
}

// (a1) clusters per slice
__global__ void __launch_bounds__(A1_THREADS) k_slice_count(Dev d, SecOff so) {
  __shared__ int s_cnt[TPCCA_MAX_ROWS];
  const int base = blockIdx.x * A1_TILE;
  const int sec0 = sector_of(so, d.n_sectors, min(base, d.n - 1));  // the block's first sector is privatised
  for (int r = threadIdx.x; r < d.n_rows; r += A1_THREADS) s_cnt[r] = 0;
  __syncthreads();
  bool bad = false;
#pragma unroll
  for (int k = 0; k < A1_ITEMS; k++) {
    const int i = base + k * A1_THREADS + threadIdx.x;
    if (i >= d.n) continue;
    const float4 c = __ldg(&d.clusters[i]);
    const int row = __float_as_int(c.w);
    if (row < 0 || row >= d.n_rows || !cluster_finite(c)) { bad = true; continue; }
    if (i < so.v[sec0 + 1]) atomicAdd(&s_cnt[row], 1);
    else atomicAdd(&d.slice_count[sector_of(so, d.n_sectors, i) * d.n_rows + row], 1);
  }
  if (bad) atomicOr(&d.cnt->status, TPCCA_STAT_BAD_CLUSTER);
  __syncthreads();
  for (int r = threadIdx.x; r < d.n_rows; r += A1_THREADS)
    if (s_cnt[r]) atomicAdd(&d.slice_count[sec0 * d.n_rows + r], s_cnt[r]);
}

// (a2) slice offsets, bin offsets (upper-bound layout), fill cursors, per-row constants of the neighbours finder
__global__ void __launch_bounds__(1024) k_slice_offsets(Dev d) {
  __shared__ int sm[32];
  int carry_c = 0, carry_b = 0;
  for (int b0 = 0; b0 < d.n_slices; b0 += 1024) {
    const int sl = b0 + threadIdx.x;
    int cnt = 0, cap = 0;
    if (sl < d.n_slices) {
      cnt = d.slice_count[sl];
      cap = (int)((float)cnt * d.P.grid_bins_per_cluster) + 129;
    }
    int tot_c, tot_b;
    const int ec = block_scan_excl(cnt, &tot_c, sm);
    const int eb = block_scan_excl(cap, &tot_b, sm);
    if (sl < d.n_slices) {
      d.row_start[sl] = carry_c + ec;
      d.slice_fill[sl] = carry_c + ec;
      d.bin_base[sl] = carry_b + eb;
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
        nb.wyu = fmaf(dxu, d.P.nbr_dydx, d.P.nbr_margin_y);
        nb.wzu = fmaf(dxu, d.P.nbr_dzdx, d.P.nbr_margin_z);
        nb.wyd = fmaf(dxd, d.P.nbr_dydx, d.P.nbr_margin_y);
        nb.wzd = fmaf(dxd, d.P.nbr_dzdx, d.P.nbr_margin_z);
      }
      d.nbr[sl] = nb;
    }
    carry_c += tot_c;
    carry_b += tot_b;
  }
  if (threadIdx.x == 0) {
    d.row_start[d.n_slices] = carry_c;
    d.bin_base[d.n_slices] = carry_b;
  }
}

// (a3) scatter into slice order: records (y, z, input index); clears the selector's hit weights on the way
__global__ void __launch_bounds__(A1_THREADS) k_slice_scatter(Dev d, SecOff so) {
  __shared__ int s_cnt[TPCCA_MAX_ROWS], s_base[TPCCA_MAX_ROWS];
  const int base = blockIdx.x * A1_TILE;
  const int sec0 = sector_of(so, d.n_sectors, min(base, d.n - 1));
  for (int r = threadIdx.x; r < d.n_rows; r += A1_THREADS) s_cnt[r] = 0;
  __syncthreads();
  float4 c[A1_ITEMS];
  int rank[A1_ITEMS];  // >= 0: rank inside the block's (sec0, row) run; -1: other sector; -2: skipped
#pragma unroll
  for (int k = 0; k < A1_ITEMS; k++) {
    const int i = base + k * A1_THREADS + threadIdx.x;
    rank[k] = -2;
    if (i >= d.n) continue;
    d.hit_weight[i] = 0ull;
    c[k] = __ldg(&d.clusters[i]);
    const int row = __float_as_int(c[k].w);
    if (row < 0 || row >= d.n_rows || !cluster_finite(c[k])) { d.out_assign[i] = -1; continue; }
    rank[k] = (i < so.v[sec0 + 1]) ? atomicAdd(&s_cnt[row], 1) : -1;
  }
  __syncthreads();
  for (int r = threadIdx.x; r < d.n_rows; r += A1_THREADS)
    if (s_cnt[r]) s_base[r] = atomicAdd(&d.slice_fill[sec0 * d.n_rows + r], s_cnt[r]);
  __syncthreads();
#pragma unroll
  for (int k = 0; k < A1_ITEMS; k++) {
    if (rank[k] == -2) continue;
    const int i = base + k * A1_THREADS + threadIdx.x;
    const int row = __float_as_int(c[k].w);
    int pos;
    if (rank[k] >= 0) pos = s_base[row] + rank[k];
    else pos = atomicAdd(&d.slice_fill[sector_of(so, d.n_sectors, i) * d.n_rows + row], 1);
    d.srec[pos] = make_float4(c[k].y, c[k].z, __int_as_float(i), 0.0f);
  }
}

// (a4) one block per slice: bounding box -> grid header -> bin histogram -> exclusive scan -> scatter
#ifndef A4_THREADS
#define A4_THREADS 512
#endif
#ifndef A4_SMEM_BINS
#define A4_SMEM_BINS 12288
#endif
// A4_SMEM_BINS bins are held in shared memory (48 KB: four 512-thread blocks per SM); a larger slice keeps its
// counters in bin_start itself

__device__ __forceinline__ int bin_of(const GridHdr& g, float y, float z) {
  int by = (int)((y - g.ymin) * g.inv_by);
  int bz = (int)((z - g.zmin) * g.inv_bz);
  by = max(0, min(by, g.ny - 1));
  bz = max(0, min(bz, g.nz - 1));
  return by * g.nz + bz;
}

__global__ void __launch_bounds__(A4_THREADS) k_slice_sort(Dev d) {
  extern __shared__ int s_hist[];
  __shared__ int sm[32];
  __shared__ uint32_t s_box[4];
  const int sl = blockIdx.x, tid = threadIdx.x;
  const int b = d.row_start[sl], e = d.row_start[sl + 1], cnt = e - b;
  const int bbase = d.bin_base[sl];
  GridHdr g;
  g.ymin = g.zmin = 0.0f; g.inv_by = g.inv_bz = 0.0f; g.ny = g.nz = 1; g.bin_base = bbase; g.pad = 0;
  if (cnt == 0) {
    if (tid == 0) d.grid[sl] = g;
    return;
  }
  // ---- bounding box (ordered-uint min / max)
  if (tid < 4) s_box[tid] = (tid & 1) ? 0u : 0xFFFFFFFFu;
  __syncthreads();
  {
    uint32_t ylo = 0xFFFFFFFFu, yhi = 0u, zlo = 0xFFFFFFFFu, zhi = 0u;
    for (int i = b + tid; i < e; i += A4_THREADS) {
      const float4 c = d.srec[i];
      const uint32_t oy = ordf(c.x), oz = ordf(c.y);
      ylo = min(ylo, oy); yhi = max(yhi, oy); zlo = min(zlo, oz); zhi = max(zhi, oz);
    }
    ylo = __reduce_min_sync(0xffffffffu, ylo); yhi = __reduce_max_sync(0xffffffffu, yhi);
    zlo = __reduce_min_sync(0xffffffffu, zlo); zhi = __reduce_max_sync(0xffffffffu, zhi);
    if ((tid & 31) == 0) {
      atomicMin(&s_box[0], ylo); atomicMax(&s_box[1], yhi); atomicMin(&s_box[2], zlo); atomicMax(&s_box[3], zhi);
    }
  }
  __syncthreads();
  // ---- grid header (every thread computes the same values)
  {
    const float ymin = unordf(s_box[0]), ymax = unordf(s_box[1]), zmin = unordf(s_box[2]), zmax = unordf(s_box[3]);
    const float ye = fmaxf(ymax - ymin, 1e-3f), ze = fmaxf(zmax - zmin, 1e-3f);
    int ny = (int)fminf(ye / d.P.grid_bin_y, 127.0f) + 1;  // clamped before the cast: a huge y extent cannot overflow
    const float want = (float)cnt * d.P.grid_bins_per_cluster / (float)ny;
    int nz = (int)want + 1;
    const int nz_cap = (int)fminf(ze / d.P.grid_bin_z_min, 1.0e6f) + 1;
    nz = max(1, min(nz, nz_cap));
    if (ny * nz + 1 > d.bin_base[sl + 1] - bbase) { ny = 1; nz = 1; }  // cannot happen: ny*nz <= bins_per_cluster*cnt + 128
    g.ymin = ymin; g.zmin = zmin;
    g.inv_by = ((float)ny / ye) * 0.9999f;
    g.inv_bz = ((float)nz / ze) * 0.9999f;
    g.ny = ny; g.nz = nz; g.pad = cnt;
  }
  const int nb = g.ny * g.nz;
  // counters: hist[k] = count -> start -> end of bin k; bin_start[bbase + 1 + k] receives end(k) = start(k + 1)
  int* hist = (nb <= A4_SMEM_BINS) ? s_hist : (d.bin_start + bbase + 1);
  for (int k = tid; k < nb; k += A4_THREADS) hist[k] = 0;
  __syncthreads();
  for (int i = b + tid; i < e; i += A4_THREADS) {
    const float4 c = d.srec[i];
    atomicAdd(&hist[bin_of(g, c.x, c.y)], 1);
  }
  __syncthreads();
  if (nb <= A4_SMEM_BINS) {  // exclusive scan in place (+ b); shared memory: thread t owns an odd-length run of bins
    const int chunk = ((nb + A4_THREADS - 1) / A4_THREADS) | 1;
    const int k0 = min(tid * chunk, nb), k1 = min(k0 + chunk, nb);
    int s = 0;
    for (int k = k0; k < k1; k++) s += hist[k];
    int tot;
    int ex = block_scan_excl(s, &tot, sm) + b;
    for (int k = k0; k < k1; k++) {
      const int v = hist[k];
      hist[k] = ex;
      ex += v;
    }
  } else {  // global memory: one tile of A4_THREADS bins per step (coalesced)
    int carry = b;
    for (int k0 = 0; k0 < nb; k0 += A4_THREADS) {
      const int k = k0 + tid;
      const int v = (k < nb) ? hist[k] : 0;
      int tot;
      const int ex = block_scan_excl(v, &tot, sm);
      if (k < nb) hist[k] = carry + ex;
      carry += tot;
    }
  }
  __syncthreads();
  for (int i = b + tid; i < e; i += A4_THREADS) {
    const float4 c = d.srec[i];
    const int pos = atomicAdd(&hist[bin_of(g, c.x, c.y)], 1);
    d.yz[pos] = make_float2(c.x, c.y);
    d.orig_idx[pos] = __float_as_int(c.z);
    d.slice_of[pos] = (uint16_t)sl;
  }
  __syncthreads();
  if (nb <= A4_SMEM_BINS)
    for (int k = tid; k < nb; k += A4_THREADS) d.bin_start[bbase + 1 + k] = hist[k];
  if (tid == 0) {
    d.bin_start[bbase] = b;
    d.grid[sl] = g;
    d.slice_bbox[4 * sl + 0] = s_box[0]; d.slice_bbox[4 * sl + 1] = s_box[1];
    d.slice_bbox[4 * sl + 2] = s_box[2]; d.slice_bbox[4 * sl + 3] = s_box[3];
    atomicAdd(&d.cnt->n_bins, nb);
  }
}

cudaError_t setup_grid_kernels() {
  return cudaFuncSetAttribute(k_slice_sort, cudaFuncAttributeMaxDynamicSharedMemorySize, A4_SMEM_BINS * (int)sizeof(int));
}

void launch_grid(const Dev& d, const SecOff& so, Launch& L) {
  k_reset<<<32, 256, 0, L.st>>>(d);
  L.count++;
  if (d.n > 0) {
    k_slice_count<<<(d.n + A1_TILE - 1) / A1_TILE, A1_THREADS, 0, L.st>>>(d, so);
    L.count++;
  }
  k_slice_offsets<<<1, 1024, 0, L.st>>>(d);
  L.count++;
  if (d.n > 0) {
    KTIMED(L, TPCCA_K_SLICE_SCATTER, (k_slice_scatter<<<(d.n + A1_TILE - 1) / A1_TILE, A1_THREADS, 0, L.st>>>(d, so)));
    L.count++;
  }
  KTIMED(L, TPCCA_K_SLICE_SORT, (k_slice_sort<<<d.n_slices, A4_THREADS, A4_SMEM_BINS * sizeof(int), L.st>>>(d)));
  L.count++;
}
