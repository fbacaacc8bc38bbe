// tpcca_merge.cu -- sector-segment merger and final fit (steps O8-O10).
// PAPER.md:51 "The second phase merges the track segments found in the individual sectors and performs the final track fit
// with the full Kalman filter"; :69 rejection of outliers by predicted chi2; :70 enlarged errors for shared clusters;
// :71 inward, outward, inward.  Works on what the last tpcca_track left in the workspace: the track records, the outer
// ends written by k_refit, the owned-hit lists of k_select_own and the shared-cluster flags.
#include "tpcca_dev.cuh"

#define M_NONE 0xffffffffffffffffull

// ---------------------------------------------------------------- (m0) reset, candidate buckets, shared flags of the lists
// The inner ends are bucketed by (sector, first_row) with a counting sort (histogram -> scan -> scatter), so that the row
// window of DESIGN.md B2 is ONE contiguous range of the sorted order.  Scratch: the per-slice arrays of the grid and
// start-hit steps (slice_nstart / slice_sbase / slice_fill), free once tpcca_track is through.
__global__ void __launch_bounds__(256) k_merge_reset(Dev d) {
  const int nt = d.cnt->n_tracks;
  const int i = blockIdx.x * blockDim.x + threadIdx.x;
  if (i == 0) { d.cnt->n_merged = 0; d.cnt->n_links = 0; d.cnt->n_fit_failed = 0; }
  // counting-sort scratch of the fit order (slot 4): strided, the grid may be smaller than the slot (small capacities)
  for (int j = i; j < 1024; j += gridDim.x * blockDim.x) d.ord[4 * 1024 + j] = 0;
  if (i <= d.n_slices) d.slice_nstart[i] = 0;
  if (i < nt) {
    d.m_best_out[i] = M_NONE; d.m_best_in[i] = M_NONE;
    d.m_next[i] = -1; d.m_prev[i] = -1;
    d.track_merged_out[i] = -1;  // stays -1 only for a segment no head reaches (cannot happen for ring != 1; k_leg_tags checks)
  }
}
__global__ void __launch_bounds__(256) k_merge_count(Dev d) {
  const int t = blockIdx.x * blockDim.x + threadIdx.x;
  if (t >= d.cnt->n_tracks) return;
  const int4 ti = *reinterpret_cast<const int4*>(&d.out_tracks[t]);  // sector, first_row, last_row, n_hits
  if (d.out_tracks[t].ndf >= 0) atomicAdd(&d.slice_nstart[ti.x * d.n_rows + ti.y], 1);
}
__global__ void __launch_bounds__(1024) k_merge_offsets(Dev d) {
  __shared__ int sm[32];
  int carry = 0;
  for (int b0 = 0; b0 < d.n_slices; b0 += 1024) {
    const int sl = b0 + threadIdx.x;
    const int v = (sl < d.n_slices) ? d.slice_nstart[sl] : 0;
    int tot;
    const int e = block_scan_excl(v, &tot, sm);
    if (sl < d.n_slices) { d.slice_sbase[sl] = carry + e; d.slice_fill[sl] = carry + e; }
    carry += tot;
  }
  if (threadIdx.x == 0) d.slice_sbase[d.n_slices] = carry;
}
__global__ void __launch_bounds__(256) k_merge_scatter(Dev d) {
  const int t = blockIdx.x * blockDim.x + threadIdx.x;
  if (t >= d.cnt->n_tracks) return;
  const tpcca_track_rec& T = d.out_tracks[t];
  if (T.ndf < 0) return;
  const int pos = atomicAdd(&d.slice_fill[T.sector * d.n_rows + T.first_row], 1);
  d.m_cand[pos] = make_int2(__float_as_int(T.z), t);  // order inside a bucket is arbitrary: the match takes min (chi2, id)
}

__global__ void __launch_bounds__(256) k_merge_shared(Dev d) {  // list entry -> shared flag of its cluster
  const unsigned long long n = d.cnt->track_hits;
  for (unsigned long long j = blockIdx.x * (unsigned long long)blockDim.x + threadIdx.x; j < n;
       j += (unsigned long long)gridDim.x * blockDim.x)
    d.th_shared[j] = d.shared_flag[d.th_hit[j]];
}

// ---------------------------------------------------------------- (m1) matching: one warp per outer end
// The lanes walk the inner ends of the neighbouring sector inside the row window (one contiguous range of m_cand, read
// coalesced: z and id); a lane whose candidate passes the z window evaluates the match (frame change, transport, chi2).
// best_out by a warp reduction, best_in by atomicMin of (chi2 bits << 32 | id): min chi2, then lower id (B4).
__global__ void __launch_bounds__(128) k_merge_match(Dev d) {
  const int lane = threadIdx.x & 31;
  const int a = (blockIdx.x * 128 + threadIdx.x) >> 5;
  if (a >= d.cnt->n_tracks) return;
  const tpcca_track_rec* tr = d.out_tracks;
  if (tr[a].ndf < 0) return;
  const float4* oa = reinterpret_cast<const float4*>(d.track_outer + (size_t)a * 24);
  const float4 o0 = oa[0];  // x, y, z, sinphi
  const float th = d.tan_half_angle;
  if (!(fabsf(o0.y) >= fmaf(o0.x, th, -d.MP.merge_edge_dist))) return;
  const int side = o0.y > 0.0f ? 1 : -1;
  const int sb = ring_neighbour(tr[a].sector, side, d.MP.ring);
  if (sb < 0 || sb >= d.n_sectors) return;
  const int last_row = tr[a].last_row;
  const int r_lo = max(0, last_row - d.MP.merge_row_back), r_hi = min(d.n_rows - 1, last_row + d.MP.merge_row_fwd);
  if (r_lo > r_hi) return;
  const float za = o0.z;
  const Rot R = sector_rotation(th);
  unsigned long long best = M_NONE;
  const int b0 = d.slice_sbase[sb * d.n_rows + r_lo], b1 = d.slice_sbase[sb * d.n_rows + r_hi + 1];
  for (int bb = b0; bb < b1; bb += 32) {
    const int pos = bb + lane;
    if (pos >= b1) continue;
    const int2 cz = d.m_cand[pos];
    if (!(fabsf(__int_as_float(cz.x) - za) <= d.MP.merge_dz_max)) continue;
    const int b = cz.y;
    const tpcca_track_rec& B = tr[b];
    KF k;
    const float4 o1 = oa[1], o2 = oa[2], o3 = oa[3], o4 = oa[4];
    k.x = o0.x; k.y = o0.y; k.z = 0.0f; k.s = o0.w; k.t = o1.x; k.q = o1.y;
    k.c00 = o1.z; k.c10 = o1.w; k.c11 = o2.x; k.c20 = o2.y; k.c21 = o2.z; k.c22 = o2.w;
    k.c30 = o3.x; k.c31 = o3.y; k.c32 = o3.z; k.c33 = o3.w; k.c40 = o4.x; k.c41 = o4.y; k.c42 = o4.z; k.c43 = o4.w;
    k.c44 = d.track_outer[(size_t)a * 24 + 20];
    k.chi2 = 0.0f;
    if (!kf_rotate(k, R.ca, (float)side * R.sa, d.kq, d.P.max_sinphi)) continue;
    if (!kf_transport(k, B.x, d.kq, d.P.max_sinphi)) continue;
    float dd = k.y - B.y;
    float chi = (dd * dd) / (k.c00 + B.cov[0]);
    dd = k.z - (B.z - za);
    chi = chi + (dd * dd) / (k.c11 + B.cov[2]);
    dd = k.s - B.sinphi;
    chi = chi + (dd * dd) / (k.c22 + B.cov[5]);
    dd = k.t - B.dzds;
    chi = chi + (dd * dd) / (k.c33 + B.cov[9]);
    dd = k.q - B.qpt;
    chi = chi + (dd * dd) / (k.c44 + B.cov[14]);
    if (!(chi <= d.MP.merge_chi2_cut)) continue;
    const unsigned long long cb = (unsigned long long)__float_as_uint(chi) << 32;  // chi >= +0: bits order like values
    best = min(best, cb | (unsigned)b);
    atomicMin(&d.m_best_in[b], cb | (unsigned)a);
  }
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) {
    const unsigned long long v = __shfl_xor_sync(0xffffffffu, best, o);
    best = min(best, v);
  }
  if (lane == 0) d.m_best_out[a] = best;
}

// ---------------------------------------------------------------- (m2) mutual links, heads
__global__ void __launch_bounds__(256) k_merge_link(Dev d) {
  const int a = blockIdx.x * blockDim.x + threadIdx.x;
  if (a >= d.cnt->n_tracks) return;
  const unsigned long long bo = d.m_best_out[a];
  if (bo == M_NONE) return;
  const int b = (int)(bo & 0xffffffffull);
  const unsigned long long bi = d.m_best_in[b];
  if (bi != M_NONE && (int)(bi & 0xffffffffull) == a) {
    d.m_next[a] = b;
    d.m_prev[b] = a;
    atomicAdd(&d.cnt->n_links, 1);
  }
}
__global__ void __launch_bounds__(256) k_merge_heads(Dev d) {
  const int t = blockIdx.x * blockDim.x + threadIdx.x;
  const int nt = d.cnt->n_tracks;
  if (t < nt) d.m_scan[t] = d.m_prev[t] < 0 ? 1 : 0;
}
// (m3) after the scan: merged id of every head; the head walks its chain (<= 20 segments) and labels the segments
__global__ void __launch_bounds__(256) k_merge_chains(Dev d) {
  const int t = blockIdx.x * blockDim.x + threadIdx.x;
  const int nt = d.cnt->n_tracks;
  if (t == 0) d.cnt->n_merged = d.m_scan[nt];
  if (t >= nt || d.m_prev[t] >= 0) return;
  const int mid = d.m_scan[t];
  d.m_head[mid] = t;
  int len = 0;
  for (int s = t; s >= 0; s = d.m_next[s]) {
    d.track_merged_out[s] = mid;
    len += d.out_tracks[s].n_hits;
  }
  d.m_len[mid] = len >> 1;  // work-order key of the fit (0..256 after clamping)
}

// ---------------------------------------------------------------- (m4) final fit: one lane per merged track, longest first
#define MERGE_MAX_SEGS 24
__global__ void __launch_bounds__(64) k_merge_fit(Dev d) {
  const int p = blockIdx.x * blockDim.x + threadIdx.x;
  if (p >= d.cnt->n_merged) return;
  const int mid = d.m_order[p];
  const int head = d.m_head[mid];
  const tpcca_track_rec* tr = d.out_tracks;
  int segs[MERGE_MAX_SEGS];
  int n_seg = 0, n = 0;
  int s_rest = head;
  for (; s_rest >= 0 && n_seg < MERGE_MAX_SEGS; s_rest = d.m_next[s_rest]) { segs[n_seg++] = s_rest; n += tr[s_rest].n_hits; }
  if (s_rest >= 0) atomicOr(&d.cnt->status, TPCCA_STAT_CHAIN_TRUNCATED);  // never with the default cuts (>= 8 rows gained per segment)
  const int last = segs[n_seg - 1];
  const Rot R = sector_rotation(d.tan_half_angle);
  // start: chord of the two outermost hits of the outermost segment, q/pT of its record
  const int2 wl_last = d.w_list[d.track_w[last]];
  const float2 pN = d.th_yz[wl_last.x + wl_last.y - 1], pM = d.th_yz[wl_last.x + wl_last.y - 2];
  const int rN = d.th_row[wl_last.x + wl_last.y - 1], rM = d.th_row[wl_last.x + wl_last.y - 2];
  const float z_ref = pN.y;
  KF k;
  {
    const float dx = d.row_x[rN] - d.row_x[rM], dy = pN.x - pM.x, dz = pN.y - pM.y;
    const float ds = sqrtf(fmaf(dx, dx, dy * dy));
    k.x = d.row_x[rN];
    k.y = pN.x; k.z = 0.0f; k.s = dy / ds; k.t = dz / ds; k.q = tr[last].qpt;
  }
  const float ey1 = d.P.sigma_y * d.MP.shared_err_scale, ez1 = d.P.sigma_z * d.MP.shared_err_scale;
  const float vy_sh = ey1 * ey1, vz_sh = ez1 * ez1;
  bool ok = true;
  int n_used = 0, n_shared = 0;
  int cur_sec = tr[last].sector;
  for (int pass = 0; pass < 3 && ok; pass++) {
    kf_reset_cov(k, d.P.cov0);
    n_used = 0; n_shared = 0;
    for (int si = 0; si < n_seg && ok; si++) {
      const int seg = (pass == 1) ? segs[si] : segs[n_seg - 1 - si];
      const int2 wl = d.w_list[d.track_w[seg]];
      const int sec = tr[seg].sector;
      if (sec != cur_sec) {  // adjacent sectors by construction of the chain
        const int sgn = (ring_neighbour(cur_sec, +1, d.MP.ring) == sec) ? 1 : -1;
        if (!kf_rotate(k, R.ca, (float)sgn * R.sa, d.kq, d.P.max_sinphi)) { ok = false; break; }
        cur_sec = sec;
      }
      for (int i = 0; i < wl.y; i++) {
        const int j = wl.x + ((pass == 1) ? i : wl.y - 1 - i);
        const float2 pj = d.th_yz[j];
        const int r = d.th_row[j];
        const bool sh = d.th_shared[j] != 0;
        if (!kf_transport(k, d.row_x[r], d.kq, d.P.max_sinphi)) { ok = false; break; }
        const float vy = sh ? vy_sh : d.sy2, vz = sh ? vz_sh : d.sz2;
        n_shared += sh ? 1 : 0;
        const float iy = 1.0f / (k.c00 + vy), iz = 1.0f / (k.c11 + vz);
        const float dy = pj.x - k.y;
        const float dz = (pj.y - z_ref) - k.z;
        const float dist = fmaf(dz * dz, iz, (dy * dy) * iy);
        if (!(dist <= d.MP.fit_reject_cut)) continue;  // outlier for this pass
        kf_update(k, pj.x, pj.y - z_ref, vy, vz, iy);
        n_used++;
      }
    }
  }
  tpcca_track_rec o;
  const tpcca_track_rec H = tr[head];
  if (ok) {
    o.x = k.x; o.y = k.y; o.z = k.z + z_ref; o.sinphi = k.s; o.dzds = k.t; o.qpt = k.q;
    o.cov[0] = k.c00; o.cov[1] = k.c10; o.cov[2] = k.c11; o.cov[3] = k.c20; o.cov[4] = k.c21; o.cov[5] = k.c22;
    o.cov[6] = k.c30; o.cov[7] = k.c31; o.cov[8] = k.c32; o.cov[9] = k.c33; o.cov[10] = k.c40; o.cov[11] = k.c41;
    o.cov[12] = k.c42; o.cov[13] = k.c43; o.cov[14] = k.c44;
    o.chi2 = k.chi2;
    o.ndf = 2 * n_used - 5;
  } else {  // keep the innermost segment's own fit, flagged (B6)
    o = H;
    o.ndf = -1;
    atomicAdd(&d.cnt->n_fit_failed, 1);
  }
  o.sector = H.sector; o.first_row = H.first_row; o.last_row = tr[last].last_row; o.n_hits = n;
  o.pad[0] = n_seg; o.pad[1] = tr[last].sector; o.pad[2] = ok ? n - n_used : -1; o.pad[3] = n_shared; o.pad[4] = head;
  float4* dst = reinterpret_cast<float4*>(&d.merged_out[mid]);
  const float4* src = reinterpret_cast<const float4*>(&o);
#pragma unroll
  for (int i = 0; i < 8; i++) dst[i] = src[i];
}

__global__ void k_merge_header(Dev d) {
  tpcca_out_header hd;
  hd.n_tracks = d.cnt->n_merged; hd.n_tracklets = d.cnt->n_links; hd.n_start_hits = d.cnt->n_fit_failed;
  hd.status = d.cnt->status;
  *d.merged_hdr = hd;
}

void launch_merge(const Dev& d, Launch& L) {
  const int K = d.max_tracks;
  if (d.n > 0 && K > 0) {
    const int nb = (max(K, d.n_slices + 1) + 255) / 256;
    k_merge_reset<<<nb, 256, 0, L.st>>>(d);
    k_merge_count<<<(K + 255) / 256, 256, 0, L.st>>>(d);
    k_merge_offsets<<<1, 1024, 0, L.st>>>(d);
    k_merge_scatter<<<(K + 255) / 256, 256, 0, L.st>>>(d);
    k_merge_shared<<<d.n_sm * 8, 256, 0, L.st>>>(d);
    k_merge_match<<<(K + 3) / 4, 128, 0, L.st>>>(d);
    k_merge_link<<<(K + 255) / 256, 256, 0, L.st>>>(d);
    k_merge_heads<<<(K + 255) / 256, 256, 0, L.st>>>(d);
    L.count += 8;
    launch_scan_i32(d.m_scan, &d.cnt->n_tracks, K, d.scan_tmp, L);
    k_merge_chains<<<(K + 255) / 256, 256, 0, L.st>>>(d);
    L.count++;
    launch_order_desc(d, 4, d.m_len, &d.cnt->n_merged, K, d.m_order, L);
    k_merge_fit<<<(K + 63) / 64, 64, 0, L.st>>>(d);
    L.count++;
  }
  k_merge_header<<<1, 1, 0, L.st>>>(d);
  L.count++;
}

// ---------------------------------------------------------------- z / time estimate (step O11)
// The helix of a fitted state is a circle in the xy plane (centre left of the direction by 1/k, k = q kq); the point of
// the circle nearest to the beam line lies on the line origin -> centre.  Turning angle from the state to that point:
// atan2(-sg (c x + s y), R - sg (s x - c y)) (no cancellation for stiff tracks), path length = angle / k.
__device__ __forceinline__ tpcca_time_rec time_estimate(const tpcca_track_rec& T, float kq, float zmin_hits, float zmax_hits,
                                                        int side, float vdrift, float z_max) {
  const float x = T.x, y = T.y, s = T.sinphi, c = sqrtf(1.0f - s * s), k = T.qpt * kq;
  float ds, dca;
  if (fabsf(k) < 1e-9f) {
    ds = -(c * x + s * y);
    dca = y * c - x * s;
  } else {
    const float R = 1.0f / fabsf(k), sg = k > 0.0f ? 1.0f : -1.0f;
    const float dphi = atan2f(-sg * (c * x + s * y), R - sg * (s * x - c * y));
    ds = dphi / k;
    const float xc = x - s / k, yc = y + c / k;
    const float Rc = sqrtf(xc * xc + yc * yc);
    dca = sg * ((x * x + y * y + 2.0f * sg * R * (y * c - x * s)) / (Rc + R));  // sg (Rc - R) without the cancellation
  }
  tpcca_time_rec o;
  const float zd = T.z + T.dzds * ds;
  const float lo = side > 0 ? zmax_hits - z_max : zmax_hits;
  const float hi = side > 0 ? zmin_hits : zmin_hits + z_max;
  float sh = zd;
  if (sh > hi) sh = hi;
  if (sh < lo) sh = lo;
  o.z_dca = zd; o.z_shift = sh; o.t0_us = (float)side * sh / vdrift; o.dca_xy = dca;
  return o;
}

__global__ void __launch_bounds__(128) k_time_estimate(Dev d, int merged, float vdrift, float z_max,
                                                        tpcca_time_rec* __restrict__ out) {
  const int i = blockIdx.x * blockDim.x + threadIdx.x;
  const int n = merged ? d.cnt->n_merged : d.cnt->n_tracks;
  if (i >= n) return;
  const tpcca_track_rec T = merged ? d.merged_out[i] : d.out_tracks[i];
  float zmin = 3.0e38f, zmax = -3.0e38f;
  for (int t = merged ? T.pad[4] : i; t >= 0; t = merged ? d.m_next[t] : -1) {
    const int2 wl = d.w_list[d.track_w[t]];
    for (int j = 0; j < wl.y; j++) {
      const float z = d.th_yz[wl.x + j].y;
      zmin = fminf(zmin, z); zmax = fmaxf(zmax, z);
    }
  }
  const int half = d.n_sectors / 2;
  const int side = (half > 0 && T.sector >= half) ? -1 : 1;
  out[i] = time_estimate(T, d.kq, zmin, zmax, side, vdrift, z_max);
}

void launch_time_estimate(const Dev& d, float vdrift, float z_max, tpcca_time_rec* out_sector, tpcca_time_rec* out_merged,
                          Launch& L) {
  if (d.n <= 0 || d.max_tracks <= 0) return;
  const int nb = (d.max_tracks + 127) / 128;
  if (out_sector) { k_time_estimate<<<nb, 128, 0, L.st>>>(d, 0, vdrift, z_max, out_sector); L.count++; }
  if (out_merged) { k_time_estimate<<<nb, 128, 0, L.st>>>(d, 1, vdrift, z_max, out_merged); L.count++; }
}
