// tpcca_select_fit.cu -- steps (f) tracklet selector and (g) final refit, plus the intermediate exports.
// (f) north_star (f): shared clusters go to the longest / best tracklet (packed weight, O6);
//     PAPER.md:55 (low clone rate), :70 (shared clusters).
// (g) PAPER.md:71 "The final Kalman refit is iterated three times: inward, outward, and inward" (O7).
#include "tpcca_dev.cuh"

// ---------------------------------------------------------------- (f1) ownership -> accept flag + packed hit list
// One warp per surviving seed w: lanes take consecutive rows (coalesced row_hit reads, 32 independent weight
// gathers).  An accepted tracklet's owned hits are packed innermost-first into th_yz / th_row at a slot range
// taken from a bump allocator (every hit has one owner, so all lists together hold at most n entries).
#define SEL_THREADS 128
#define SEL_CHUNKS (TPCCA_MAX_ROWS / 32)
__global__ void __launch_bounds__(SEL_THREADS) k_select_own(Dev d) {
  const unsigned lane = threadIdx.x & 31;
  const int n_work = d.cnt->n_work, n_warps = (gridDim.x * SEL_THREADS) >> 5;
  for (int w = (blockIdx.x * SEL_THREADS + threadIdx.x) >> 5; w < n_work; w += n_warps) {
    const int t = d.work_t[w];
    const int4 ti = reinterpret_cast<const int4*>(d.tl_ints)[t];
    if (!ti.x) continue;
    const unsigned long long W = d.tl_W[t];
    const int32_t* rh = d.row_hit + (size_t)w * d.n_rows;
    int hh[SEL_CHUNKS];
    unsigned mm[SEL_CHUNKS];
    int owned = 0;
#pragma unroll
    for (int c = 0; c < SEL_CHUNKS; c++) {
      const int r = ti.y + 32 * c + (int)lane;
      int h = -1;
      if (r <= ti.z) h = rh[r];
      const bool own = (h >= 0) && (d.hit_weight[h] == W);
      hh[c] = own ? h : -1;
      mm[c] = __ballot_sync(0xffffffffu, own);
      owned += __popc(mm[c]);
    }
    if (owned < d.P.min_track_hits) continue;
    // accepted: the hits this tracklet collected but lost to another owner are shared clusters (B7)
#pragma unroll
    for (int c = 0; c < SEL_CHUNKS; c++) {
      const int r = ti.y + 32 * c + (int)lane;
      if (hh[c] < 0 && r <= ti.z) {
        const int h = rh[r];
        if (h >= 0) d.shared_flag[h] = 1;
      }
    }
    int off = 0;
    if (lane == 0) off = (int)atomicAdd(&d.cnt->track_hits, (unsigned long long)owned);
    off = __shfl_sync(0xffffffffu, off, 0);
    int base = off;
#pragma unroll
    for (int c = 0; c < SEL_CHUNKS; c++) {
      if (hh[c] >= 0) {
        const int j = base + __popc(mm[c] & ((1u << lane) - 1u));
        d.th_yz[j] = d.yz[hh[c]];
        d.th_row[j] = (uint8_t)(ti.y + 32 * c + (int)lane);
        d.th_hit[j] = hh[c];
      }
      base += __popc(mm[c]);
    }
    if (lane == 0) {
      d.sel_scan[t] = 1;
      d.w_list[w] = make_int2(off, owned);
    }
  }
}

// ---------------------------------------------------------------- (f2) after the scan: track ids, length histogram
// Track ids follow tracklet-id order (the work list is in that order).
__global__ void __launch_bounds__(256) k_select_ids(Dev d) {
  const int w = blockIdx.x * blockDim.x + threadIdx.x;
  const int nw = d.cnt->n_work;
  if (w == 0) {
    const int tot = d.sel_scan[d.cnt->n_start];
    if (tot > d.max_tracks) atomicOr(&d.cnt->status, TPCCA_STAT_TRACK_OVERFLOW);
    d.cnt->n_tracks = min(tot, d.max_tracks);
  }
  if (w >= nw) return;
  const int t = d.work_t[w];
  const int id = d.sel_scan[t];
  const bool acc = (d.sel_scan[t + 1] != id) && (id < d.max_tracks);
  d.tl_track[t] = acc ? id : -1;
  if (acc) {
    d.track_w[id] = w;
    d.track_tracklet[id] = t;
    d.track_len[id] = d.w_list[w].y;
  }
}

// ---------------------------------------------------------------- (f3) cluster -> track assignment
__global__ void __launch_bounds__(256) k_assign(Dev d) {
  const int h = blockIdx.x * blockDim.x + threadIdx.x;
  if (h >= d.row_start[d.n_slices]) return;
  const unsigned long long w = d.hit_weight[h];
  int tr = -1;
  if (w) {
    const uint32_t tid = 0xFFFFFFFFu - (uint32_t)(w & 0xFFFFFFFFull);
    tr = d.tl_track[tid];
  }
  d.out_assign[d.orig_idx[h]] = tr;
}

void launch_select(const Dev& d, Launch& L) {
  if (d.n <= 0 || d.max_tracklets <= 0) return;
  const int T = d.max_tracklets;
  KTIMED(L, TPCCA_K_SELECT_OWN, (k_select_own<<<d.n_sm * 16, SEL_THREADS, 0, L.st>>>(d)));
  L.count++;
  launch_scan_i32(d.sel_scan, &d.cnt->n_start, T, d.scan_tmp, L);
  k_select_ids<<<(T + 255) / 256, 256, 0, L.st>>>(d);
  KTIMED(L, TPCCA_K_ASSIGN, (k_assign<<<(d.n + 255) / 256, 256, 0, L.st>>>(d)));
  L.count += 2;
  // refit order: tracks by decreasing hit count, so that the lanes of a refit warp run the same number of steps
  launch_order_desc(d, 0, d.track_len, &d.cnt->n_tracks, d.max_tracks, d.track_order, L);
}

// ---------------------------------------------------------------- (g) refit
// One thread per track, tracks taken in decreasing-length order; a track's hits are one contiguous list.
__global__ void __launch_bounds__(64) k_refit(Dev d) {
  const int p = blockIdx.x * blockDim.x + threadIdx.x;
  if (p >= d.cnt->n_tracks) return;
  const int id = d.track_order[p];
  const int w = d.track_w[id];
  const int2 wl = d.w_list[w];
  const int n_hits = wl.y;
  const int t = d.track_tracklet[id];
  const int sector = d.slice_of[d.start_hits[t]] / d.n_rows;
  const float q0 = d.tl_floats[8 * t + 5];
  const float2* ly = d.th_yz + wl.x;
  const uint8_t* lr = d.th_row + wl.x;
  const int rN = lr[n_hits - 1], rM = lr[n_hits - 2], r_in = lr[0];
  const float2 pN = ly[n_hits - 1], pM = ly[n_hits - 2];
  const float z_ref = pN.y;
  KF k;
  {
    const float dx = d.row_x[rN] - d.row_x[rM], dy = pN.x - pM.x, dz = pN.y - pM.y;
    const float ds = sqrtf(fmaf(dx, dx, dy * dy));
    k.x = d.row_x[rN];
    k.y = pN.x; k.z = 0.0f; k.s = dy / ds; k.t = dz / ds; k.q = q0;
  }
  bool ok = true, outer_written = false;
  for (int pass = 0; pass < 3 && ok; pass++) {
    kf_reset_cov(k, d.P.cov0);
    for (int i = 0; i < n_hits; i++) {
      const int j = (pass == 1) ? i : n_hits - 1 - i;
      const float2 pj = ly[j];
      const int r = lr[j];
      if (!kf_transport(k, d.row_x[r], d.kq, d.P.max_sinphi)) { ok = false; break; }
      kf_update(k, pj.x, pj.y - z_ref, d.sy2, d.sz2);
    }
    if (pass == 1 && ok) {  // end of the outward pass: the outer end of the track (O8), kept for tpcca_merge
      float4* od = reinterpret_cast<float4*>(d.track_outer + (size_t)id * 24);
      od[0] = make_float4(k.x, k.y, k.z + z_ref, k.s);
      od[1] = make_float4(k.t, k.q, k.c00, k.c10);
      od[2] = make_float4(k.c11, k.c20, k.c21, k.c22);
      od[3] = make_float4(k.c30, k.c31, k.c32, k.c33);
      od[4] = make_float4(k.c40, k.c41, k.c42, k.c43);
      od[5] = make_float4(k.c44, 0.f, 0.f, 0.f);
      outer_written = true;
    }
  }
  if (!outer_written) {  // the refit failed before the outward pass ended: no outer end (the merger skips ndf < 0)
    float4* od = reinterpret_cast<float4*>(d.track_outer + (size_t)id * 24);
    for (int i = 0; i < 6; i++) od[i] = make_float4(0.f, 0.f, 0.f, 0.f);
  }
  tpcca_track_rec o;
  o.sector = sector;
  o.first_row = r_in; o.last_row = rN; o.n_hits = n_hits;
  o.x = k.x; o.y = k.y; o.z = k.z + z_ref; o.sinphi = k.s; o.dzds = k.t; o.qpt = k.q;
  o.cov[0] = k.c00; o.cov[1] = k.c10; o.cov[2] = k.c11; o.cov[3] = k.c20; o.cov[4] = k.c21; o.cov[5] = k.c22;
  o.cov[6] = k.c30; o.cov[7] = k.c31; o.cov[8] = k.c32; o.cov[9] = k.c33; o.cov[10] = k.c40; o.cov[11] = k.c41;
  o.cov[12] = k.c42; o.cov[13] = k.c43; o.cov[14] = k.c44;
  o.chi2 = k.chi2;
  o.ndf = ok ? 2 * n_hits - 5 : -1;
  for (int i = 0; i < 5; i++) o.pad[i] = 0;
  float4* dst = reinterpret_cast<float4*>(&d.out_tracks[id]);
  const float4* src = reinterpret_cast<const float4*>(&o);
#pragma unroll
  for (int i = 0; i < 8; i++) dst[i] = src[i];
}

__global__ void k_write_header(Dev d) {
  tpcca_out_header hd;
  hd.n_tracks = d.cnt->n_tracks; hd.n_tracklets = d.cnt->n_valid; hd.n_start_hits = d.cnt->n_start;
  hd.status = d.cnt->status;
  *d.out_hdr = hd;
}

void launch_refit(const Dev& d, Launch& L) {
  if (d.n > 0 && d.max_tracks > 0) {
    KTIMED(L, TPCCA_K_REFIT, (k_refit<<<(d.max_tracks + 63) / 64, 64, 0, L.st>>>(d)));
    L.count++;
  }
  k_write_header<<<1, 1, 0, L.st>>>(d);
  L.count++;
}

// ---------------------------------------------------------------- exports (input-index space)
__global__ void k_export_links(Dev d, int what, int32_t* dst) {
  const int h = blockIdx.x * blockDim.x + threadIdx.x;
  if (h >= d.row_start[d.n_slices]) return;
  int v;
  if (what == TPCCA_LINK_UP_RAW) v = d.link_up[h];
  else if (what == TPCCA_LINK_DOWN_RAW) v = d.link_down[h];
  else if (what == TPCCA_LINK_UP) v = d.link_up_clean[h];
  else {
    v = d.link_down[h];
    if (v >= 0 && d.link_up[v] != h) v = -1;
  }
  dst[d.orig_idx[h]] = (v >= 0) ? d.orig_idx[v] : -1;
}
__global__ void k_export_fill(Dev d, int32_t* dst) {  // clusters ignored by the grid (bad row)
  const int i = blockIdx.x * blockDim.x + threadIdx.x;
  if (i < d.n) dst[i] = -1;
}
__global__ void k_export_tracklets(Dev d, int what, void* dst) {
  const int t = blockIdx.x * blockDim.x + threadIdx.x;
  if (t >= d.cnt->n_start) return;
  if (what == TPCCA_START_HITS) ((int32_t*)dst)[t] = d.orig_idx[d.start_hits[t]];
  else if (what == TPCCA_TRACKLET_INTS) ((int4*)dst)[t] = reinterpret_cast<const int4*>(d.tl_ints)[t];
  else if (what == TPCCA_TRACKLET_FLOATS) {
    ((float4*)dst)[2 * t] = reinterpret_cast<const float4*>(d.tl_floats)[2 * t];
    ((float4*)dst)[2 * t + 1] = reinterpret_cast<const float4*>(d.tl_floats)[2 * t + 1];
  } else if (what == TPCCA_TRACKLET_ROW_HITS) {
    const int4 ti = reinterpret_cast<const int4*>(d.tl_ints)[t];
    int32_t* o = (int32_t*)dst + (size_t)t * d.n_rows;
    for (int r = 0; r < d.n_rows; r++) {
      int v = -1;
      if (ti.x && r >= ti.y && r <= ti.z) {
        v = d.row_hit[(size_t)d.seed_w[t] * d.n_rows + r];
        if (v >= 0) v = d.orig_idx[v];
      }
      o[r] = v;
    }
  }
}
__global__ void k_export_track_tracklet(Dev d, int what, int32_t* dst) {
  const int i = blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= d.cnt->n_tracks) return;
  if (what == TPCCA_TRACK_TRACKLET) dst[i] = d.track_tracklet[i];
  else if (what == TPCCA_MERGE_LINK_NEXT) dst[i] = d.m_next[i];
  else {
    const float4* src = reinterpret_cast<const float4*>(d.track_outer + (size_t)i * 24);
    float4* o = reinterpret_cast<float4*>(dst) + (size_t)i * 6;
    for (int q = 0; q < 6; q++) o[q] = src[q];
  }
}
__global__ void k_export_shared(Dev d, int32_t* dst) {
  const int h = blockIdx.x * blockDim.x + threadIdx.x;
  if (h < d.row_start[d.n_slices]) dst[d.orig_idx[h]] = d.shared_flag[h];
}

void launch_export(const Dev& d, int what, void* dst, Launch& L) {
  if (what <= TPCCA_LINK_DOWN) {
    if (d.n <= 0) return;
    k_export_fill<<<(d.n + 255) / 256, 256, 0, L.st>>>(d, (int32_t*)dst);
    k_export_links<<<(d.n + 255) / 256, 256, 0, L.st>>>(d, what, (int32_t*)dst);
  } else if (what == TPCCA_TRACK_TRACKLET || what == TPCCA_MERGE_LINK_NEXT || what == TPCCA_TRACK_OUTER) {
    if (d.max_tracks > 0) k_export_track_tracklet<<<(d.max_tracks + 255) / 256, 256, 0, L.st>>>(d, what, (int32_t*)dst);
  } else if (what == TPCCA_SHARED) {
    if (d.n <= 0) return;
    k_export_fill<<<(d.n + 255) / 256, 256, 0, L.st>>>(d, (int32_t*)dst);  // ignored clusters: -1
    k_export_shared<<<(d.n + 255) / 256, 256, 0, L.st>>>(d, (int32_t*)dst);
  } else {
    if (d.max_tracklets > 0) k_export_tracklets<<<(d.max_tracklets + 127) / 128, 128, 0, L.st>>>(d, what, dst);
  }
}
