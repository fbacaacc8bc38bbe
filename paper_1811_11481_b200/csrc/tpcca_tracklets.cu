// tpcca_tracklets.cu -- step (e): tracklet constructor (north_star (e); O5).
// PAPER.md:51  seeds "fit with a simplified Kalman Filter ... extrapolated through the TPC volume,
//              adjacent hits are collected without following multiple track hypotheses, and the fit is refined";
// PAPER.md:65-68  outward first, then inward through the seed rejecting outliers;
// PAPER.md:57  parallel over tracks;  PAPER.md:121  fp32, z kept relative to the start hit.
// One thread per start hit.  E1 seed fit along the links, E2 outward pick-up, E3 inward pass.
#include "tpcca_dev.cuh"

// Best pick-up candidate of slice `sl` for the predicted state; sorted index or -1.  (O5 "search")
__device__ __forceinline__ int search_row(const Dev& d, int sl, const KF& k, float z_ref, float cut) {
  const int rb = d.row_start[sl], re = d.row_start[sl + 1];
  if (re <= rb) return -1;
  const float vy = k.c00 + d.sy2, vz = k.c11 + d.sz2;
  const float iy = 1.0f / vy, iz = 1.0f / vz;
  const float wy = sqrtf(cut * vy), wz = sqrtf(cut * vz);
  const GridHdr g = d.grid[sl];
  const float zc = z_ref + k.z;  // search centre in frame coordinates (bin lookup only)
  const float mz = 2e-3f + (fabsf(zc) + fabsf(z_ref) + fabsf(k.z)) * 4e-7f;
  int y0, y1, z0, z1;
  bin_range(k.y - wy - 1e-3f, k.y + wy + 1e-3f, g.ymin, g.inv_by, g.ny, y0, y1);
  bin_range(zc - wz - mz, zc + wz + mz, g.zmin, g.inv_bz, g.nz, z0, z1);
  int best = -1;
  float bd = 0.0f, by = 0.0f, bz = 0.0f;
  if (z0 > z1) return -1;
  for (int yb = y0; yb <= y1; yb++) {
    const int cb = d.bin_start[g.bin_base + yb * g.nz + z0];
    const int ce = d.bin_start[g.bin_base + yb * g.nz + z1 + 1];
    for (int c = cb; c < ce; c++) {
      const float2 p = d.yz[c];
      const float dy = p.x - k.y;
      const float dz = (p.y - z_ref) - k.z;
      if (!(fabsf(dy) <= wy) || !(fabsf(dz) <= wz)) continue;
      const float dist = (dy * dy) * iy + (dz * dz) * iz;
      if (!(dist <= cut)) continue;
      bool better;
      if (best < 0) better = true;
      else if (dist != bd) better = dist < bd;
      else better = key_less(p.y, p.x, d.orig_idx[c], bz, by, d.orig_idx[best]);
      if (better) { best = c; bd = dist; by = p.x; bz = p.y; }
    }
  }
  return best;
}

__device__ __forceinline__ unsigned long long pack_weight(const Dev& d, int n_hits, float chi2, uint32_t tid) {
  float qf = (d.P.qual_scale * chi2) / (float)(2 * n_hits);
  qf = fminf(65535.0f, qf);
  qf = fmaxf(0.0f, qf);
  const int qi = (int)qf;
  const uint32_t qual = (uint32_t)(65535 - qi);
  return ((unsigned long long)(uint32_t)n_hits << 48) | ((unsigned long long)qual << 32) |
         (unsigned long long)(0xFFFFFFFFu - tid);
}

#define E_THREADS 64
__global__ void __launch_bounds__(E_THREADS) k_tracklets(Dev d) {
  const int t = blockIdx.x * blockDim.x + threadIdx.x;
  if (t >= d.cnt->n_start) return;
  const int T = d.max_tracklets;
  const int R = d.n_rows;
  int32_t* rh = d.row_hit + t;  // rh[r * T]
  const int h0 = d.start_hits[t];
  const int sl0 = d.slice_of[h0];
  const int sec = sl0 / R, r0 = sl0 - sec * R;
  const int sbase = sec * R;
  int4 ti = make_int4(0, -1, -1, 0);
  float4 tf0 = make_float4(0.f, 0.f, 0.f, 0.f), tf1 = make_float4(0.f, 0.f, 0.f, 0.f);
  unsigned long long W = 0ull;
  int n_steps = 0, n_search = 0;  // work counters (roofline units)

  const float2 p0 = d.yz[h0];
  const float z_ref = p0.y;
  tf1.w = z_ref;
  KF k;
  bool ok = true;
  int last_row = r0, n_chain = 1;
  {  // E1: seed fit along the cleaned up-links
    int h = d.link_up_clean[h0];
    int r = (h >= d.row_start[sbase + r0 + 2]) ? r0 + 2 : r0 + 1;
    const float2 p1 = d.yz[h];
    const float dx = d.row_x[r] - d.row_x[r0], dy = p1.x - p0.x, dz = p1.y - p0.y;
    const float ds = sqrtf(dx * dx + dy * dy);
    k.x = d.row_x[r0];
    k.y = p0.x; k.z = 0.0f; k.s = dy / ds; k.t = dz / ds; k.q = 0.0f;
    kf_reset_cov(k, d.P.cov0);
    kf_update(k, p0.x, p0.y - z_ref, d.sy2, d.sz2);
    rh[(size_t)r0 * T] = h0;
    while (h >= 0) {
      const float2 p = d.yz[h];
      n_steps++;
      if (!kf_transport(k, d.row_x[r], d.kq, d.P.max_sinphi)) { ok = false; break; }
      kf_update(k, p.x, p.y - z_ref, d.sy2, d.sz2);
      if (r == last_row + 2) rh[(size_t)(r - 1) * T] = -1;  // skipped (empty) row
      rh[(size_t)r * T] = h;
      last_row = r;
      n_chain++;
      h = d.link_up_clean[h];
      if (h >= 0) r = (r + 2 < R && h >= d.row_start[sbase + r + 2]) ? r + 2 : r + 1;
    }
    if (n_chain < d.P.min_seed_hits) ok = false;
  }
  if (ok) {
    // E2: outward extrapolation, one best cluster per row
    float sx = k.x, sy = k.y, sz = k.z, ss = k.s, st = k.t, sq = k.q;  // snapshot at the outermost hit
    int top_row = last_row, gap = 0;
    for (int r = last_row + 1; r < R; r++) {
      n_steps++;
      if (!kf_transport(k, d.row_x[r], d.kq, d.P.max_sinphi)) break;
      if (fabsf(k.y) > d.row_x[r] * d.tan_half_angle + d.P.edge_margin) break;
      n_search++;
      const int hb = search_row(d, sbase + r, k, z_ref, d.P.pick_cut);
      rh[(size_t)r * T] = hb;
      if (hb >= 0) {
        const float2 p = d.yz[hb];
        kf_update(k, p.x, p.y - z_ref, d.sy2, d.sz2);
        gap = 0; top_row = r;
        sx = k.x; sy = k.y; sz = k.z; ss = k.s; st = k.t; sq = k.q;
      } else {
        gap++;
        if (gap > d.P.max_gap) break;
      }
    }
    // E3: inward pass through the seed with outlier rejection, then pick-up below it
    k.x = sx; k.y = sy; k.z = sz; k.s = ss; k.t = st; k.q = sq;
    kf_reset_cov(k, d.P.cov0);
    KF inner = k;
    int inner_row = -1, n_hits = 0, outer_row = -1;
    gap = 0;
    for (int r = top_row; r >= 0; r--) {
      n_steps++;
      if (!kf_transport(k, d.row_x[r], d.kq, d.P.max_sinphi)) break;
      if (fabsf(k.y) > d.row_x[r] * d.tan_half_angle + d.P.edge_margin) break;
      bool hit = false;
      const int cur = (r >= r0) ? rh[(size_t)r * T] : -1;
      if (cur >= 0) {
        const float2 p = d.yz[cur];
        const float iy = 1.0f / (k.c00 + d.sy2), iz = 1.0f / (k.c11 + d.sz2);
        const float dy = p.x - k.y;
        const float dz = (p.y - z_ref) - k.z;
        const float dist = (dy * dy) * iy + (dz * dz) * iz;
        if (dist <= d.P.reject_cut) { kf_update(k, p.x, p.y - z_ref, d.sy2, d.sz2); hit = true; }
        else rh[(size_t)r * T] = -1;
      } else {
        n_search++;
        const int hb = search_row(d, sbase + r, k, z_ref, d.P.pick_cut);
        rh[(size_t)r * T] = hb;
        if (hb >= 0) {
          const float2 p = d.yz[hb];
          kf_update(k, p.x, p.y - z_ref, d.sy2, d.sz2);
          hit = true;
        }
      }
      if (hit) {
        gap = 0; inner = k; inner_row = r; n_hits++;
        if (outer_row < 0) outer_row = r;
      } else {
        gap++;
        if (r < r0 && gap > d.P.max_gap) break;
      }
    }
    // rows below inner_row hold no accepted hit: consumers only read [first_row, last_row]
    if (inner_row >= 0 && n_hits >= d.P.min_tracklet_hits) {
      ti = make_int4(1, inner_row, outer_row, n_hits);
      tf0 = make_float4(inner.x, inner.y, inner.z, inner.s);
      tf1 = make_float4(inner.t, inner.q, inner.chi2, z_ref);
      W = pack_weight(d, n_hits, inner.chi2, (uint32_t)t);
      for (int r = inner_row; r <= outer_row; r++) {
        const int h = rh[(size_t)r * T];
        if (h >= 0) atomicMax(&d.hit_weight[h], W);
      }
      atomicAdd(&d.cnt->n_valid, 1);
    }
  }
  {
    const unsigned m = __activemask();
    const int ws = __reduce_add_sync(m, n_steps), wq = __reduce_add_sync(m, n_search);
    if ((threadIdx.x & 31) == (__ffs(m) - 1)) {
      atomicAdd(&d.cnt->row_steps, (unsigned long long)ws);
      atomicAdd(&d.cnt->searches, (unsigned long long)wq);
    }
  }
  reinterpret_cast<int4*>(d.tl_ints)[t] = ti;
  reinterpret_cast<float4*>(d.tl_floats)[2 * t] = tf0;
  reinterpret_cast<float4*>(d.tl_floats)[2 * t + 1] = tf1;
  d.tl_W[t] = W;
}

void launch_tracklets(const Dev& d, Launch& L) {
  if (d.n <= 0 || d.max_tracklets <= 0) return;
  k_tracklets<<<(d.max_tracklets + E_THREADS - 1) / E_THREADS, E_THREADS, 0, L.st>>>(d);
  L.count++;
}
