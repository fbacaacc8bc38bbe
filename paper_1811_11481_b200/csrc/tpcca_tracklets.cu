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

// ---------------------------------------------------------------- (e0) seed filter + stable compaction
// A start hit whose link chain is shorter than min_seed_hits is void (O5/E1) and never reaches
// the constructor: the survivors are compacted in tracklet-id order into the work list (w -> t).
__global__ void __launch_bounds__(256) k_seed_flag(Dev d) {
  const int t = blockIdx.x * blockDim.x + threadIdx.x;
  if (t >= d.cnt->n_start) return;
  int h = d.start_hits[t], n = 1;
  while (n < d.P.min_seed_hits) {
    h = d.link_up_clean[h];
    if (h < 0) break;
    n++;
  }
  const int keep = n >= d.P.min_seed_hits ? 1 : 0;
  d.seed_w[t] = keep;
  if (!keep) {
    reinterpret_cast<int4*>(d.tl_ints)[t] = make_int4(0, -1, -1, 0);
    reinterpret_cast<float4*>(d.tl_floats)[2 * t] = make_float4(0.f, 0.f, 0.f, 0.f);
    reinterpret_cast<float4*>(d.tl_floats)[2 * t + 1] = make_float4(0.f, 0.f, 0.f, 0.f);
    d.tl_W[t] = 0ull;
  }
}

__global__ void __launch_bounds__(256) k_seed_compact(Dev d) {
  const int t = blockIdx.x * blockDim.x + threadIdx.x;
  const int ns = d.cnt->n_start;
  if (t == 0) d.cnt->n_work = d.seed_w[ns];
  if (t >= ns) return;
  const int w = d.seed_w[t];
  if (d.seed_w[t + 1] != w) d.work_t[w] = t;
}

// ---------------------------------------------------------------- (e) constructor
// Persistent warps: every lane runs one seed at a time and, when it is done, takes the next one from a
// global queue (one atomic per warp refill, ballot + popc ranks), so a warp never idles on its longest
// tracklet.  E1 (follow links), E2 (outward pick-up) and E3 (inward pass) run as ONE loop with a phase
// variable, so lanes in different phases share the single transport / search / update instruction streams.
// row_hit is [w][row]: a lane's consecutive rows fall into the same 32-byte sector, which L2 merges.
#define E_THREADS 128
#define E_BLOCKS_PER_SM 6
#define PH_E1 0
#define PH_E2 1
#define PH_E3 2
#define PH_DONE 3

__global__ void __launch_bounds__(E_THREADS, E_BLOCKS_PER_SM) k_tracklets(Dev d) {
  const int R = d.n_rows;
  const int n_work = d.cnt->n_work;
  const unsigned lane = threadIdx.x & 31;
  int n_steps = 0, n_search = 0, n_val = 0;  // work counters (roofline units)
  // per-seed state
  int t = -1, r0 = 0, sbase = 0, h = -1, r = 0;
  int32_t* rh = nullptr;
  float z_ref = 0.f;
  KF k;
  k.x = 0.f; k.y = k.z = k.s = k.t = k.q = 0.f; kf_reset_cov(k, d.P.cov0);
  int phase = PH_DONE;
  bool exhausted = false, valid = true;
  int last_row = 0, top_row = 0, gap = 0;
  float sx = 0.f, sy = 0.f, sz = 0.f, ss = 0.f, st = 0.f, sq = 0.f;             // snapshot at the outermost hit
  float ix = 0.f, iy_ = 0.f, iz_ = 0.f, is = 0.f, it = 0.f, iq = 0.f, ichi = 0.f;  // state at the innermost hit
  int inner_row = -1, outer_row = -1, n_hits = 0;

  while (true) {
    const bool need = (phase == PH_DONE) && !exhausted;
    const unsigned need_mask = __ballot_sync(0xffffffffu, need);
    if (need_mask) {
      if (need && t >= 0) {  // retire the finished seed
        int4 ti = make_int4(0, -1, -1, 0);
        float4 tf0 = make_float4(0.f, 0.f, 0.f, 0.f), tf1 = make_float4(0.f, 0.f, 0.f, z_ref);
        unsigned long long W = 0ull;
        if (valid && inner_row >= 0 && n_hits >= d.P.min_tracklet_hits) {
          ti = make_int4(1, inner_row, outer_row, n_hits);
          tf0 = make_float4(ix, iy_, iz_, is);
          tf1 = make_float4(it, iq, ichi, z_ref);
          W = pack_weight(d, n_hits, ichi, (uint32_t)t);
          n_val++;
        }
        reinterpret_cast<int4*>(d.tl_ints)[t] = ti;
        reinterpret_cast<float4*>(d.tl_floats)[2 * t] = tf0;
        reinterpret_cast<float4*>(d.tl_floats)[2 * t + 1] = tf1;
        d.tl_W[t] = W;
        t = -1;
      }
      int base = 0;
      const int leader = __ffs(need_mask) - 1;
      if ((int)lane == leader) base = atomicAdd(&d.cnt->work_next, __popc(need_mask));
      base = __shfl_sync(0xffffffffu, base, leader);
      if (need) {
        const int w = base + __popc(need_mask & ((1u << lane) - 1u));
        if (w >= n_work) exhausted = true;
        else {  // start seed w (E1 initial state: DESIGN.md O5)
          t = d.work_t[w];
          rh = d.row_hit + (size_t)w * R;
          const int h0 = d.start_hits[t];
          const int sl0 = d.slice_of[h0];
          const int sec = sl0 / R;
          r0 = sl0 - sec * R;
          sbase = sec * R;
          const float2 p0 = d.yz[h0];
          z_ref = p0.y;
          h = d.link_up_clean[h0];
          r = (h >= d.row_start[sbase + r0 + 2]) ? r0 + 2 : r0 + 1;
          const float2 p1 = d.yz[h];
          const float dx = d.row_x[r] - d.row_x[r0], dy = p1.x - p0.x, dz = p1.y - p0.y;
          const float ds = sqrtf(dx * dx + dy * dy);
          k.x = d.row_x[r0];
          k.y = p0.x; k.z = 0.0f; k.s = dy / ds; k.t = dz / ds; k.q = 0.0f;
          kf_reset_cov(k, d.P.cov0);
          kf_update(k, p0.x, p0.y - z_ref, d.sy2, d.sz2);
          rh[r0] = h0;
          phase = PH_E1; valid = true;
          last_row = r0; top_row = r0; gap = 0;
          inner_row = -1; outer_row = -1; n_hits = 0;
        }
      }
      if (__ballot_sync(0xffffffffu, !exhausted) == 0u) break;
    }
    if (phase == PH_DONE) continue;  // exhausted lane: idle until the warp is finished

    // ---- one row step
    n_steps++;
    const float xr = d.row_x[r];
    const bool tr_ok = kf_transport(k, xr, d.kq, d.P.max_sinphi);
    const bool edge = (phase != PH_E1) && (fabsf(k.y) > xr * d.tan_half_angle + d.P.edge_margin);
    const bool stop = !tr_ok || edge;
    int cand = -1;
    bool accept = false, do_search = false;
    float2 pc = make_float2(0.f, 0.f);
    if (!stop) {
      if (phase == PH_E1) {
        cand = h; accept = true;
      } else {
        const int cur = (phase == PH_E3 && r >= r0) ? rh[r] : -1;
        if (cur >= 0) {
          cand = cur;
          pc = d.yz[cur];
          const float iy = 1.0f / (k.c00 + d.sy2), iz = 1.0f / (k.c11 + d.sz2);
          const float dy = pc.x - k.y;
          const float dz = (pc.y - z_ref) - k.z;
          const float dist = (dy * dy) * iy + (dz * dz) * iz;
          accept = dist <= d.P.reject_cut;
          if (!accept) rh[r] = -1;
        } else {
          do_search = true;
        }
      }
    }
    if (do_search) {
      n_search++;
      cand = search_row(d, sbase + r, k, z_ref, d.P.pick_cut);
      rh[r] = cand;
      accept = cand >= 0;
    }
    if (accept) {
      if (phase == PH_E1 || do_search) pc = d.yz[cand];
      kf_update(k, pc.x, pc.y - z_ref, d.sy2, d.sz2);
    }
    // ---- bookkeeping and phase transitions
    bool to_e3 = false;
    if (phase == PH_E1) {
      if (stop) { valid = false; phase = PH_DONE; }
      else {
        if (r == last_row + 2) rh[r - 1] = -1;  // skipped (empty) row
        rh[r] = h;
        last_row = r;
        h = d.link_up_clean[h];
        if (h >= 0) r = (r + 2 < R && h >= d.row_start[sbase + r + 2]) ? r + 2 : r + 1;
        else {  // seed complete (its length was checked by k_seed_flag): start E2
          phase = PH_E2; top_row = last_row; gap = 0;
          sx = k.x; sy = k.y; sz = k.z; ss = k.s; st = k.t; sq = k.q;
          r = last_row + 1;
          if (r >= R) to_e3 = true;
        }
      }
    } else if (phase == PH_E2) {
      if (stop) to_e3 = true;
      else {
        if (accept) { gap = 0; top_row = r; sx = k.x; sy = k.y; sz = k.z; ss = k.s; st = k.t; sq = k.q; }
        else { gap++; if (gap > d.P.max_gap) to_e3 = true; }
        r++;
        if (r >= R) to_e3 = true;
      }
    } else {  // PH_E3
      if (stop) phase = PH_DONE;
      else {
        if (accept) {
          gap = 0; inner_row = r; n_hits++;
          if (outer_row < 0) outer_row = r;
          ix = k.x; iy_ = k.y; iz_ = k.z; is = k.s; it = k.t; iq = k.q; ichi = k.chi2;
        } else {
          gap++;
          if (r < r0 && gap > d.P.max_gap) phase = PH_DONE;
        }
        r--;
        if (r < 0) phase = PH_DONE;
      }
    }
    if (to_e3) {  // restore the state at the outermost hit, reset the covariance, go inward through the seed
      k.x = sx; k.y = sy; k.z = sz; k.s = ss; k.t = st; k.q = sq;
      kf_reset_cov(k, d.P.cov0);
      gap = 0; r = top_row; phase = PH_E3;
    }
  }
  const int ws = __reduce_add_sync(0xffffffffu, n_steps), wq = __reduce_add_sync(0xffffffffu, n_search),
            wv = __reduce_add_sync(0xffffffffu, n_val);
  if (lane == 0 && ws) {
    atomicAdd(&d.cnt->row_steps, (unsigned long long)ws);
    atomicAdd(&d.cnt->searches, (unsigned long long)wq);
    atomicAdd(&d.cnt->n_valid, wv);
  }
}

// (e2) every hit of a valid tracklet receives max(weight) (O5 "Result")
__global__ void __launch_bounds__(128) k_tracklet_weights(Dev d) {
  const int w = blockIdx.x * blockDim.x + threadIdx.x;
  if (w >= d.cnt->n_work) return;
  const int t = d.work_t[w];
  const int4 ti = reinterpret_cast<const int4*>(d.tl_ints)[t];
  if (!ti.x) return;
  const unsigned long long W = d.tl_W[t];
  const int32_t* rh = d.row_hit + (size_t)w * d.n_rows;
  for (int r = ti.y; r <= ti.z; r++) {
    const int h = rh[r];
    if (h >= 0) atomicMax(&d.hit_weight[h], W);
  }
}

void launch_tracklets(const Dev& d, Launch& L) {
  if (d.n <= 0 || d.max_tracklets <= 0) return;
  const int T = d.max_tracklets;
  k_seed_flag<<<(T + 255) / 256, 256, 0, L.st>>>(d);
  L.count++;
  launch_scan_i32(d.seed_w, &d.cnt->n_start, T, d.scan_tmp, L);
  k_seed_compact<<<(T + 255) / 256, 256, 0, L.st>>>(d);
  k_tracklets<<<148 * E_BLOCKS_PER_SM, E_THREADS, 0, L.st>>>(d);
  k_tracklet_weights<<<(T + 127) / 128, 128, 0, L.st>>>(d);
  L.count += 3;
}
