// tpcca_select_fit.cu -- steps (f) tracklet selector and (g) final refit, plus the intermediate exports.
// (f) north_star (f): shared clusters go to the longest / best tracklet (packed weight, O6);
//     PAPER.md:55 (low clone rate), :70 (shared clusters).
// (g) PAPER.md:71 "The final Kalman refit is iterated three times: inward, outward, and inward" (O7).
#include "tpcca_dev.cuh"

// ---------------------------------------------------------------- (f1) ownership count -> accept flag
// One thread per surviving seed w.  Non-owned hits are re-encoded in place as -2-h (reversible: the
// export decodes them), so the later passes see owned hits as h >= 0.
__global__ void __launch_bounds__(128) k_select_flag(Dev d) {
  const int w = blockIdx.x * blockDim.x + threadIdx.x;
  if (w >= d.cnt->n_work) return;
  const int t = d.work_t[w];
  const int4 ti = reinterpret_cast<const int4*>(d.tl_ints)[t];
  int flag = 0;
  if (ti.x) {
    const unsigned long long W = d.tl_W[t];
    int32_t* rh = d.row_hit + (size_t)w * d.n_rows;
    int owned = 0;
    for (int r = ti.y; r <= ti.z; r++) {
      const int h = rh[r];
      if (h < 0) continue;
      if (d.hit_weight[h] == W) owned++;
      else rh[r] = -2 - h;
    }
    flag = owned >= d.P.min_track_hits ? 1 : 0;
    if (flag) atomicAdd(&d.cnt->track_hits, (unsigned long long)owned);
  }
  if (flag) d.sel_scan[t] = 1;
}

// ---------------------------------------------------------------- (f2) after the scan: track ids + packed hit lists
// Track ids follow tracklet-id order (the work list is in that order).  Each accepted track's owned hits are
// packed innermost-first into th_yz / th_row at [j][id], so that the refit's lanes read one line per step.
__global__ void __launch_bounds__(128) k_select_write(Dev d) {
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
  if (!acc) return;
  const int4 ti = reinterpret_cast<const int4*>(d.tl_ints)[t];
  const int K = d.max_tracks;
  const int32_t* rh = d.row_hit + (size_t)w * d.n_rows;
  int j = 0, sl = 0;
  for (int r = ti.y; r <= ti.z; r++) {
    const int h = rh[r];
    if (h < 0) continue;
    d.th_yz[(size_t)j * K + id] = d.yz[h];
    d.th_row[(size_t)j * K + id] = (uint8_t)r;
    if (j == 0) sl = d.slice_of[h];
    j++;
  }
  d.track_tracklet[id] = t;
  d.track_info[id] = j | ((sl / d.n_rows) << 16);
}

// ---------------------------------------------------------------- (f3) cluster -> track assignment
__global__ void __launch_bounds__(256) k_assign(Dev d) {
  const int h = blockIdx.x * blockDim.x + threadIdx.x;
  if (h >= d.n) return;
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
  k_select_flag<<<(T + 127) / 128, 128, 0, L.st>>>(d);
  L.count++;
  launch_scan_i32(d.sel_scan, &d.cnt->n_start, T, d.scan_tmp, L);
  k_select_write<<<(T + 127) / 128, 128, 0, L.st>>>(d);
  k_assign<<<(d.n + 255) / 256, 256, 0, L.st>>>(d);
  L.count += 2;
}

// ---------------------------------------------------------------- (g) refit
// One thread per track; hits come from the packed lists (coalesced across the warp).
__global__ void __launch_bounds__(64) k_refit(Dev d) {
  const int id = blockIdx.x * blockDim.x + threadIdx.x;
  if (id >= d.cnt->n_tracks) return;
  const int K = d.max_tracks;
  const int info = d.track_info[id];
  const int n_hits = info & 0xFFFF, sector = info >> 16;
  const int t = d.track_tracklet[id];
  const float q0 = d.tl_floats[8 * t + 5];
  const float2* ly = d.th_yz + id;
  const uint8_t* lr = d.th_row + id;
  const int rN = lr[(size_t)(n_hits - 1) * K], rM = lr[(size_t)(n_hits - 2) * K], r_in = lr[0];
  const float2 pN = ly[(size_t)(n_hits - 1) * K], pM = ly[(size_t)(n_hits - 2) * K];
  const float z_ref = pN.y;
  KF k;
  {
    const float dx = d.row_x[rN] - d.row_x[rM], dy = pN.x - pM.x, dz = pN.y - pM.y;
    const float ds = sqrtf(dx * dx + dy * dy);
    k.x = d.row_x[rN];
    k.y = pN.x; k.z = 0.0f; k.s = dy / ds; k.t = dz / ds; k.q = q0;
  }
  bool ok = true;
  for (int pass = 0; pass < 3 && ok; pass++) {
    kf_reset_cov(k, d.P.cov0);
    for (int i = 0; i < n_hits; i++) {
      const int j = (pass == 1) ? i : n_hits - 1 - i;
      const float2 p = ly[(size_t)j * K];
      const int r = lr[(size_t)j * K];
      if (!kf_transport(k, d.row_x[r], d.kq, d.P.max_sinphi)) { ok = false; break; }
      kf_update(k, p.x, p.y - z_ref, d.sy2, d.sz2);
    }
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
    k_refit<<<(d.max_tracks + 63) / 64, 64, 0, L.st>>>(d);
    L.count++;
  }
  k_write_header<<<1, 1, 0, L.st>>>(d);
  L.count++;
}

// ---------------------------------------------------------------- exports (input-index space)
__global__ void k_export_links(Dev d, int what, int32_t* dst) {
  const int h = blockIdx.x * blockDim.x + threadIdx.x;
  if (h >= d.n) return;
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
        if (v <= -2) v = -2 - v;
        if (v >= 0) v = d.orig_idx[v];
      }
      o[r] = v;
    }
  }
}
__global__ void k_export_track_tracklet(Dev d, int32_t* dst) {
  const int i = blockIdx.x * blockDim.x + threadIdx.x;
  if (i < d.cnt->n_tracks) dst[i] = d.track_tracklet[i];
}

void launch_export(const Dev& d, int what, void* dst, Launch& L) {
  if (what <= TPCCA_LINK_DOWN) {
    if (d.n <= 0) return;
    k_export_fill<<<(d.n + 255) / 256, 256, 0, L.st>>>(d, (int32_t*)dst);
    k_export_links<<<(d.n + 255) / 256, 256, 0, L.st>>>(d, what, (int32_t*)dst);
  } else if (what == TPCCA_TRACK_TRACKLET) {
    if (d.max_tracks > 0) k_export_track_tracklet<<<(d.max_tracks + 255) / 256, 256, 0, L.st>>>(d, (int32_t*)dst);
  } else {
    if (d.max_tracklets > 0) k_export_tracklets<<<(d.max_tracklets + 127) / 128, 128, 0, L.st>>>(d, what, dst);
  }
}
