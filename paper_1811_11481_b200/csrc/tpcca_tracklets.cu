// tpcca_tracklets.cu -- step (e): tracklet constructor (north_star (e); O5).
// PAPER.md:51  seeds "fit with a simplified Kalman Filter ... extrapolated through the TPC volume,
//              adjacent hits are collected without following multiple track hypotheses, and the fit is refined";
// PAPER.md:65-68  outward first, then inward through the seed rejecting outliers;
// PAPER.md:57  parallel over tracks;  PAPER.md:121  fp32, z kept relative to the start hit.
// One lane per seed.  E1 seed fit along the links, E2 outward pick-up, E3a inward through the seed, E3b pick-up below it.
#include "tpcca_dev.cuh"

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
// the constructor: the survivors are compacted in tracklet-id order into the work list (w -> t), which keeps
// seeds of the same sector and row next to each other (shared grid headers and bins in L1/L2).
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
  d.sel_scan[t] = 0;
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
// Four persistent kernels, one per kind of row step of DESIGN.md O5, so that every warp runs ONE uniform step body:
//   k_tl_e1  seed fit along the links            (transport + update)
//   k_tl_e2  outward extrapolation and pick-up   (transport + search + update)
//   k_tl_e3a inward pass through the seed        (transport + keep/reject of the existing hit + update)
//   k_tl_e3b pick-up below the seed               (transport + search + update)
// Every lane runs one seed at a time and, when it is done, takes the next one from a global queue (one atomic
// per warp refill; ballot + popc give the lanes their ranks), so a warp never idles on its longest seed.
// E2, E3a and E3b take the seeds longest first (counting sort by expected row steps, launch_order_desc): with only a
// few seeds per resident lane the tail decides the time.  E1 keeps the id order: its link -> cluster gathers are local in it.
// The Kalman state travels between the kernels through tl_state[w][E_STATE].  row_hit is [w][row]: a lane's
// consecutive rows share a 32-byte sector, which L2 merges.
#ifndef E_THREADS
#define E_THREADS 128
#endif
#define E_STATE 40  // floats per seed in tl_state (layout: see k_tl_e3a)
#define FULL 0xffffffffu
#ifndef E_REFILL_MIN
#define E_REFILL_MIN 8  // refill a warp when this many lanes are idle (amortises the divergent start-up code)
#endif
#define REFILL_MIN E_REFILL_MIN

// warp-collective: lanes with need=true receive consecutive queue positions
__device__ __forceinline__ int fetch_work(int* counter, bool need, unsigned lane, unsigned need_mask) {
  int base = 0;
  const int leader = __ffs(need_mask) - 1;
  if ((int)lane == leader) base = atomicAdd(counter, __popc(need_mask));
  base = __shfl_sync(FULL, base, leader);
  return need ? base + __popc(need_mask & ((1u << lane) - 1u)) : -1;
}

__device__ __forceinline__ void st_store_kf(float* st, const KF& k) {
  float4* p = reinterpret_cast<float4*>(st);
  p[0] = make_float4(k.x, k.y, k.z, k.s);
  p[1] = make_float4(k.t, k.q, k.c00, k.c10);
  p[2] = make_float4(k.c11, k.c20, k.c21, k.c22);
  p[3] = make_float4(k.c30, k.c31, k.c32, k.c33);
  p[4] = make_float4(k.c40, k.c41, k.c42, k.c43);
  st[20] = k.c44; st[21] = k.chi2;
}
__device__ __forceinline__ void st_load_kf(const float* st, KF& k) {
  const float4* p = reinterpret_cast<const float4*>(st);
  const float4 a = p[0], b = p[1], c = p[2], e = p[3], f = p[4];
  k.x = a.x; k.y = a.y; k.z = a.z; k.s = a.w;
  k.t = b.x; k.q = b.y; k.c00 = b.z; k.c10 = b.w;
  k.c11 = c.x; k.c20 = c.y; k.c21 = c.z; k.c22 = c.w;
  k.c30 = e.x; k.c31 = e.y; k.c32 = e.z; k.c33 = e.w;
  k.c40 = f.x; k.c41 = f.y; k.c42 = f.z; k.c43 = f.w;
  k.c44 = st[20]; k.chi2 = st[21];
}

__device__ __noinline__ bool tie_less(const Dev& d, int c, float2 p, int best) {
  const float2 q = d.yz[best];
  return key_less(p.y, p.x, d.orig_idx[c], q.y, q.x, d.orig_idx[best]);
}

__device__ __forceinline__ void prefetch_l1(const void* p) { asm volatile("prefetch.global.L1 [%0];" ::"l"(p)); }

// Pick-up search of one row step (O5 "Search"): the clusters of slice g inside the window compete,
// best = min by (d, key) among d <= pick_cut.  Returns the chosen sorted index or -1; pbest = its (y, z).
// The candidates of up to two y-bin rows form one flat index space that is walked four at a time: the four loads
// are independent and every lane runs the same four evaluations, so a warp whose lanes hold 0..4 candidates
// (the usual case) makes one converged pass.
#ifndef SEARCH_UNROLL
#define SEARCH_UNROLL 3
#endif
// wy_out = 1 / (c00 + sigma_y^2): the same quotient the update of the chosen hit starts with.
__device__ __forceinline__ int search_row(const Dev& d, const GridHdr& g, const KF& k, float z_ref, float2& pbest, float& wy_out) {
  const float cut = d.P.pick_cut;
  const float vy = k.c00 + d.sy2, vz = k.c11 + d.sz2;
  const float iy = 1.0f / vy, iz = 1.0f / vz;
  wy_out = iy;
  const float wy = sqrtf(cut * vy), wz = sqrtf(cut * vz);
  int y0, y1, z0, z1;
  const float zc = z_ref + k.z;  // search centre in frame coordinates (bin lookup only)
  const float mz = 2e-3f + (fabsf(zc) + fabsf(z_ref) + fabsf(k.z)) * 4e-7f;
  bin_range_fast(k.y - wy - 1e-3f, k.y + wy + 1e-3f, g.ymin, g.inv_by, g.ny, y0, y1);
  bin_range_fast(zc - wz - mz, zc + wz + mz, g.zmin, g.inv_bz, g.nz, z0, z1);
  if (z0 > z1 || g.pad == 0) { y0 = 1; y1 = 0; }  // NaN / empty window, or empty row
  int best = -1;
  float bd = 0.0f;
  for (int yb = y0; yb <= y1; yb += 2) {
    const int* bs = d.bin_start + g.bin_base + yb * g.nz;
    const bool two = yb + 1 <= y1;
    const int a0 = bs[z0], a1 = bs[z1 + 1];
    int b0 = 0, b1 = 0;
    if (two) { b0 = bs[g.nz + z0]; b1 = bs[g.nz + z1 + 1]; }
    const int na = a1 - a0, ntot = na + (b1 - b0);
    const int jump = b0 - a1;  // flat index i >= na is cluster a0 + i + jump
    for (int i = 0; i < ntot; i += SEARCH_UNROLL) {
      float2 p[SEARCH_UNROLL];
      int c[SEARCH_UNROLL];
#pragma unroll
      for (int j = 0; j < SEARCH_UNROLL; j++) {
        const int ii = min(i + j, ntot - 1);  // clamped address; the evaluation below is predicated on i + j < ntot
        c[j] = a0 + ii + ((ii >= na) ? jump : 0);
        p[j] = d.yz[c[j]];
      }
#pragma unroll
      for (int j = 0; j < SEARCH_UNROLL; j++) {
        const float dy = p[j].x - k.y;
        const float dz = (p[j].y - z_ref) - k.z;
        const float dist = fmaf(dz * dz, iz, (dy * dy) * iy);
        const bool in = (i + j < ntot) && (fabsf(dy) <= wy) && (fabsf(dz) <= wz) && (dist <= cut);
        bool take = in && ((best < 0) || (dist < bd));
        if (in && best >= 0 && dist == bd) take = tie_less(d, c[j], p[j], best);  // exact tie: key order (rare)
        best = take ? c[j] : best;
        bd = take ? dist : bd;
        pbest.x = take ? p[j].x : pbest.x;
        pbest.y = take ? p[j].y : pbest.y;
      }
    }
  }
  return best;
}

// ---- E1: seed fit along the cleaned up-links
#ifndef E1_BLOCKS
#define E1_BLOCKS 4  // CTAs per SM in the grid: fewer lanes = more seeds per lane = better balance
#endif
#ifndef E1_BOUNDS
#define E1_BOUNDS 6
#endif
__global__ void __launch_bounds__(E_THREADS, E1_BOUNDS) k_tl_e1(Dev d) {
  const int R = d.n_rows, n_work = d.cnt->n_work;
  const unsigned lane = threadIdx.x & 31;
  int n_steps = 0;
  int w = -1, sbase = 0, h = -1, r = 0, last_row = 0;
  int hn_n = -1;                           // link of h, loaded one step ahead
  float2 pc_n = make_float2(0.f, 0.f);     // cluster h, loaded one step ahead
  int32_t* rh = nullptr;
  float z_ref = 0.f;
  KF k;
  k.x = k.y = k.z = k.s = k.t = k.q = 0.f; kf_reset_cov(k, d.P.cov0);
  bool busy = false, exhausted = false, valid = true;
  while (true) {
    const bool need = !busy && !exhausted;
    const unsigned nm = __ballot_sync(FULL, need);
    if (nm && (__popc(nm) >= REFILL_MIN || __ballot_sync(FULL, busy) == 0u)) {
      if (need && w >= 0) {  // retire
        float* st = d.tl_state + (size_t)w * E_STATE;
        st_store_kf(st, k);
        reinterpret_cast<int*>(st)[22] = last_row;
        reinterpret_cast<int*>(st)[23] = valid ? 1 : 0;
        d.e_key[w] = valid ? R - 1 - last_row : 0;  // E2 work order: rows left above the chain
        w = -1;
      }
      const int nw = fetch_work(&d.cnt->work_next[0], need, lane, nm);
      if (need) {
        if (nw >= n_work) exhausted = true;
        else {
          w = nw;
          const int t = d.work_t[w];
          rh = d.row_hit + (size_t)w * R;
          const int h0 = d.start_hits[t];
          const int sl0 = d.slice_of[h0];
          const int sec = sl0 / R, r0 = sl0 - sec * R;
          sbase = sec * R;
          const float2 p0 = d.yz[h0];
          z_ref = p0.y;
          h = d.link_up_clean[h0];
          r = (h >= d.row_start[sbase + r0 + 2]) ? r0 + 2 : r0 + 1;
          const float2 p1 = d.yz[h];
          pc_n = p1; hn_n = d.link_up_clean[h];
          const float dx = d.row_x[r] - d.row_x[r0], dy = p1.x - p0.x, dz = p1.y - p0.y;
          const float ds = sqrtf(fmaf(dx, dx, dy * dy));
          k.x = d.row_x[r0];
          k.y = p0.x; k.z = 0.0f; k.s = dy / ds; k.t = dz / ds; k.q = 0.0f;
          kf_reset_cov(k, d.P.cov0);
          kf_update(k, p0.x, p0.y - z_ref, d.sy2, d.sz2);
          rh[r0] = h0;
          last_row = r0; valid = true; busy = true;
        }
      }
      if (__ballot_sync(FULL, !exhausted) == 0u) break;
    }
    if (!busy) continue;
    // ---- one chain step.  The chain h -> link[h] -> yz[link[h]] is two dependent gathers per step; they are taken one
    // step ahead (pc, hn of THIS step were loaded during the previous one), so their latency hides behind the filter.
    n_steps++;
    const float2 pc = pc_n;
    const int hn = hn_n;
    if (hn >= 0) { pc_n = d.yz[hn]; hn_n = d.link_up_clean[hn]; }
    const int rs2 = (r + 2 < R) ? d.row_start[sbase + r + 2] : 0x7fffffff;
    if (!kf_transport(k, d.row_x[r], d.kq, d.P.max_sinphi)) { valid = false; busy = false; continue; }
    kf_update(k, pc.x, pc.y - z_ref, d.sy2, d.sz2);
    if (r == last_row + 2) rh[r - 1] = -1;  // skipped (empty) row
    rh[r] = h;
    last_row = r;
    h = hn;
    if (h < 0) busy = false;
    else r = (h >= rs2) ? r + 2 : r + 1;
  }
  const int ws = __reduce_add_sync(FULL, n_steps);
  if (lane == 0 && ws) {
    atomicAdd(&d.cnt->row_steps, (unsigned long long)ws);
    atomicAdd(&d.cnt->phase_steps[0], (unsigned long long)ws);
  }
}

// ---- E2: outward extrapolation, one best cluster per row
#ifndef E2_BLOCKS
#define E2_BLOCKS 6
#endif
__global__ void __launch_bounds__(E_THREADS, E2_BLOCKS) k_tl_e2(Dev d) {
  const int R = d.n_rows, n_work = d.cnt->n_work;
  const unsigned lane = threadIdx.x & 31;
  int n_steps = 0;
  int w = -1, sbase = 0, r = 0, r0 = 0, top_row = 0, gap = 0;
  int32_t* rh = nullptr;
  float z_ref = 0.f;
  KF k;
  k.x = k.y = k.z = k.s = k.t = k.q = 0.f; kf_reset_cov(k, d.P.cov0);
  float sx = 0.f, sy = 0.f, sz = 0.f, ss = 0.f, st_ = 0.f, sq = 0.f;  // snapshot at the outermost hit
  bool busy = false, exhausted = false, live = false;
  while (true) {
    const bool need = !busy && !exhausted;
    const unsigned nm = __ballot_sync(FULL, need);
    if (nm && (__popc(nm) >= REFILL_MIN || __ballot_sync(FULL, busy) == 0u)) {
      if (need && w >= 0) {  // retire: the snapshot replaces the state, top_row replaces last_row
        if (live) {
          float* st = d.tl_state + (size_t)w * E_STATE;
          reinterpret_cast<float4*>(st)[0] = make_float4(sx, sy, sz, ss);
          st[4] = st_; st[5] = sq;
          reinterpret_cast<int*>(st)[22] = top_row;
        }
        d.e_key[d.max_tracklets + w] = live ? top_row - r0 + 1 : 0;  // E3a work order: rows from the outermost hit down to r0
        w = -1;
      }
      const int nw = fetch_work(&d.cnt->work_next[1], need, lane, nm);
      if (need) {
        if (nw >= n_work) exhausted = true;
        else {
          w = d.e_order[nw];
          const float* st = d.tl_state + (size_t)w * E_STATE;
          live = reinterpret_cast<const int*>(st)[23] != 0;
          if (live) {
            st_load_kf(st, k);
            const int last_row = reinterpret_cast<const int*>(st)[22];
            const int t = d.work_t[w];
            const int h0 = d.start_hits[t];
            const int sl0 = d.slice_of[h0];
            sbase = (sl0 / R) * R;
            r0 = sl0 - sbase;
            z_ref = d.yz[h0].y;
            rh = d.row_hit + (size_t)w * R;
            sx = k.x; sy = k.y; sz = k.z; ss = k.s; st_ = k.t; sq = k.q;
            top_row = last_row; gap = 0; r = last_row + 1;
            busy = r < R;
          }
        }
      }
      if (__ballot_sync(FULL, !exhausted) == 0u) break;
    }
    if (!busy) continue;
    // ---- one row step
    n_steps++;
    const GridHdr g = d.grid[sbase + r];
    if (r + 1 < R) prefetch_l1(&d.grid[sbase + r + 1]);
    const float xr = d.row_x[r];
    if (!kf_transport(k, xr, d.kq, d.P.max_sinphi) || fabsf(k.y) > fmaf(xr, d.tan_half_angle, d.P.edge_margin)) {
      busy = false;
      continue;
    }
    float2 pb = make_float2(0.f, 0.f);
    float wy;
    const int cand = search_row(d, g, k, z_ref, pb, wy);
    rh[r] = cand;
    if (cand >= 0) {
      kf_update(k, pb.x, pb.y - z_ref, d.sy2, d.sz2, wy);
      gap = 0; top_row = r;
      sx = k.x; sy = k.y; sz = k.z; ss = k.s; st_ = k.t; sq = k.q;
    } else {
      gap++;
      if (gap > d.P.max_gap) busy = false;
    }
    r++;
    if (r >= R) busy = false;
  }
  const int ws = __reduce_add_sync(FULL, n_steps);
  if (lane == 0 && ws) {
    atomicAdd(&d.cnt->row_steps, (unsigned long long)ws);
    atomicAdd(&d.cnt->phase_steps[1], (unsigned long long)ws);
    atomicAdd(&d.cnt->searches, (unsigned long long)ws);
  }
}

// ---- E3: inward pass through the seed with outlier rejection, then pick-up below it.
// Two kernels so that a warp's lanes run the same kind of step:
//   k_tl_e3a  rows from the outermost hit down to the start row r0: the row already holds a hit (keep/reject test,
//             no search) except for the rare gap rows;
//   k_tl_e3b  rows below r0: every step is a pick-up search; stops after max_gap consecutive misses.
// The state crosses the boundary through tl_state[w][E_STATE] (layout below).
//   [0..21] Kalman state (st_store_kf)   [22] next row   [23] status: 0 void, 1 continue, 2 stopped (finalise only)
//   [24..30] state at the innermost accepted hit (x, y, z~, sinphi, dzds, qpt, chi2)
//   [31] inner_row  [32] outer_row  [33] n_hits  [34] gap
#ifndef E3_BLOCKS
#define E3_BLOCKS 6
#endif
#ifndef E3B_BLOCKS
#define E3B_BLOCKS 6
#endif

__global__ void __launch_bounds__(E_THREADS, E3_BLOCKS) k_tl_e3a(Dev d) {
  const int R = d.n_rows, n_work = d.cnt->n_work;
  const unsigned lane = threadIdx.x & 31;
  int n_steps = 0, n_search = 0;
  int w = -1, sbase = 0, r0 = 0, r = 0, gap = 0;
  int32_t* rh = nullptr;
  float z_ref = 0.f;
  KF k;
  k.x = k.y = k.z = k.s = k.t = k.q = 0.f; kf_reset_cov(k, d.P.cov0);
  float ix = 0.f, iy_ = 0.f, iz_ = 0.f, is = 0.f, it = 0.f, iq = 0.f, ichi = 0.f;  // state at the innermost hit
  int inner_row = -1, outer_row = -1, n_hits = 0;
  bool busy = false, exhausted = false, live = false, stopped = false;
  while (true) {
    const bool need = !busy && !exhausted;
    const unsigned nm = __ballot_sync(FULL, need);
    if (nm && (__popc(nm) >= REFILL_MIN || __ballot_sync(FULL, busy) == 0u)) {
      if (need && w >= 0) {  // retire: hand the state to k_tl_e3b
        float* st = d.tl_state + (size_t)w * E_STATE;
        int* si = reinterpret_cast<int*>(st);
        const bool cont = live && !stopped && r >= 0;
        if (live) {
          st_store_kf(st, k);
          si[22] = r;
          reinterpret_cast<float4*>(st)[6] = make_float4(ix, iy_, iz_, is);
          st[28] = it; st[29] = iq; st[30] = ichi;
          si[31] = inner_row; si[32] = outer_row; si[33] = n_hits; si[34] = gap;
        }
        si[23] = live ? (cont ? 1 : 2) : 0;
        d.e_key[2 * d.max_tracklets + w] = cont ? r + 1 : 0;  // E3b work order: rows left below the start row
        w = -1;
      }
      const int nw = fetch_work(&d.cnt->work_next[2], need, lane, nm);
      if (need) {
        if (nw >= n_work) exhausted = true;
        else {
          w = d.e_order[d.max_tracklets + nw];
          const int t = d.work_t[w];
          const float* st = d.tl_state + (size_t)w * E_STATE;
          live = reinterpret_cast<const int*>(st)[23] != 0;
          stopped = false;
          inner_row = -1; outer_row = -1; n_hits = 0; gap = 0;
          if (live) {
            const int h0 = d.start_hits[t];
            const int sl0 = d.slice_of[h0];
            const int sec = sl0 / R;
            r0 = sl0 - sec * R; sbase = sec * R;
            z_ref = d.yz[h0].y;
            const float4 a = reinterpret_cast<const float4*>(st)[0];
            k.x = a.x; k.y = a.y; k.z = a.z; k.s = a.w; k.t = st[4]; k.q = st[5];
            kf_reset_cov(k, d.P.cov0);
            r = reinterpret_cast<const int*>(st)[22];
            rh = d.row_hit + (size_t)w * R;
            busy = true;
          }
        }
      }
      if (__ballot_sync(FULL, !exhausted) == 0u) break;
    }
    if (!busy) continue;
    // ---- one row step (r >= r0).  Loads that do not depend on the filter state go first.
    n_steps++;
    const int cur = rh[r];
    float2 pb = make_float2(0.f, 0.f);
    if (cur >= 0) pb = d.yz[cur];
    const float xr = d.row_x[r];
    if (!kf_transport(k, xr, d.kq, d.P.max_sinphi) || fabsf(k.y) > fmaf(xr, d.tan_half_angle, d.P.edge_margin)) {
      busy = false; stopped = true;
      continue;
    }
    int cand;
    float wy;
    if (cur >= 0) {  // existing hit: kept iff d <= reject_cut (no window), O5/E3
      const float iy = 1.0f / (k.c00 + d.sy2), iz = 1.0f / (k.c11 + d.sz2);
      wy = iy;
      const float dy = pb.x - k.y;
      const float dz = (pb.y - z_ref) - k.z;
      const float dist = fmaf(dz * dz, iz, (dy * dy) * iy);
      cand = (dist <= d.P.reject_cut) ? cur : -1;
    } else {  // gap row inside the range (rare): pick-up search
      n_search++;
      const GridHdr g = d.grid[sbase + r];
      cand = search_row(d, g, k, z_ref, pb, wy);
    }
    if (cand != cur) rh[r] = cand;  // rejected hit -> -1, or the search result
    if (cand >= 0) {
      kf_update(k, pb.x, pb.y - z_ref, d.sy2, d.sz2, wy);
      gap = 0; inner_row = r; n_hits++;
      if (outer_row < 0) outer_row = r;
      ix = k.x; iy_ = k.y; iz_ = k.z; is = k.s; it = k.t; iq = k.q; ichi = k.chi2;
    } else {
      gap++;  // the gap stop is armed only below r0 (E3 gap rule)
    }
    r--;
    if (r < r0) busy = false;
  }
  const int ws = __reduce_add_sync(FULL, n_steps), wq = __reduce_add_sync(FULL, n_search);
  if (lane == 0 && ws) {
    atomicAdd(&d.cnt->row_steps, (unsigned long long)ws);
    atomicAdd(&d.cnt->phase_steps[2], (unsigned long long)ws);
    atomicAdd(&d.cnt->searches, (unsigned long long)wq);
  }
}

__global__ void __launch_bounds__(E_THREADS, E3B_BLOCKS) k_tl_e3b(Dev d) {
  const int R = d.n_rows, n_work = d.cnt->n_work;
  const unsigned lane = threadIdx.x & 31;
  int n_steps = 0, n_val = 0, n_vhits = 0;
  int w = -1, t = -1, sbase = 0, r = 0, gap = 0, status = 0;
  int32_t* rh = nullptr;
  float z_ref = 0.f;
  KF k;
  k.x = k.y = k.z = k.s = k.t = k.q = 0.f; kf_reset_cov(k, d.P.cov0);
  float ix = 0.f, iy_ = 0.f, iz_ = 0.f, is = 0.f, it = 0.f, iq = 0.f, ichi = 0.f;  // state at the innermost hit
  int inner_row = -1, outer_row = -1, n_hits = 0;
  bool busy = false, exhausted = false;
  while (true) {
    const bool need = !busy && !exhausted;
    const unsigned nm = __ballot_sync(FULL, need);
    if (nm && (__popc(nm) >= REFILL_MIN || __ballot_sync(FULL, busy) == 0u)) {
      if (need && w >= 0) {  // retire: tracklet record (void unless enough hits)
        int4 ti = make_int4(0, -1, -1, 0);
        float4 tf0 = make_float4(0.f, 0.f, 0.f, 0.f), tf1 = make_float4(0.f, 0.f, 0.f, z_ref);
        unsigned long long W = 0ull;
        if (status != 0 && inner_row >= 0 && n_hits >= d.P.min_tracklet_hits) {
          ti = make_int4(1, inner_row, outer_row, n_hits);
          tf0 = make_float4(ix, iy_, iz_, is);
          tf1 = make_float4(it, iq, ichi, z_ref);
          W = pack_weight(d, n_hits, ichi, (uint32_t)t);
          n_val++;
          n_vhits += n_hits;
        }
        reinterpret_cast<int4*>(d.tl_ints)[t] = ti;
        reinterpret_cast<float4*>(d.tl_floats)[2 * t] = tf0;
        reinterpret_cast<float4*>(d.tl_floats)[2 * t + 1] = tf1;
        d.tl_W[t] = W;
        w = -1;
      }
      const int nw = fetch_work(&d.cnt->work_next[3], need, lane, nm);
      if (need) {
        if (nw >= n_work) exhausted = true;
        else {
          w = d.e_order[2 * d.max_tracklets + nw];
          t = d.work_t[w];
          const float* st = d.tl_state + (size_t)w * E_STATE;
          const int* si = reinterpret_cast<const int*>(st);
          status = si[23];
          const int h0 = d.start_hits[t];
          z_ref = d.yz[h0].y;
          inner_row = -1; outer_row = -1; n_hits = 0;
          if (status != 0) {
            const float4 sn = reinterpret_cast<const float4*>(st)[6];
            ix = sn.x; iy_ = sn.y; iz_ = sn.z; is = sn.w; it = st[28]; iq = st[29]; ichi = st[30];
            inner_row = si[31]; outer_row = si[32]; n_hits = si[33];
          }
          if (status == 1) {
            st_load_kf(st, k);
            r = si[22]; gap = si[34];
            sbase = (d.slice_of[h0] / R) * R;
            rh = d.row_hit + (size_t)w * R;
            busy = true;
          }
        }
      }
      if (__ballot_sync(FULL, !exhausted) == 0u) break;
    }
    if (!busy) continue;
    // ---- one row step below the start row: transport, pick-up search, update
    n_steps++;
    const GridHdr g = d.grid[sbase + r];
    if (r > 0) prefetch_l1(&d.grid[sbase + r - 1]);
    const float xr = d.row_x[r];
    if (!kf_transport(k, xr, d.kq, d.P.max_sinphi) || fabsf(k.y) > fmaf(xr, d.tan_half_angle, d.P.edge_margin)) {
      busy = false;
      continue;
    }
    float2 pb = make_float2(0.f, 0.f);
    float wy;
    const int cand = search_row(d, g, k, z_ref, pb, wy);
    rh[r] = cand;
    if (cand >= 0) {
      kf_update(k, pb.x, pb.y - z_ref, d.sy2, d.sz2, wy);
      gap = 0; inner_row = r; n_hits++;
      if (outer_row < 0) outer_row = r;
      ix = k.x; iy_ = k.y; iz_ = k.z; is = k.s; it = k.t; iq = k.q; ichi = k.chi2;
    } else {
      gap++;
      if (gap > d.P.max_gap) busy = false;
    }
    r--;
    if (r < 0) busy = false;
  }
  const int ws = __reduce_add_sync(FULL, n_steps), wv = __reduce_add_sync(FULL, n_val);
  const int wh = __reduce_add_sync(FULL, n_vhits);
  if (lane == 0 && (ws || wv)) {
    atomicAdd(&d.cnt->row_steps, (unsigned long long)ws);
    atomicAdd(&d.cnt->phase_steps[3], (unsigned long long)ws);
    atomicAdd(&d.cnt->searches, (unsigned long long)ws);
    atomicAdd(&d.cnt->n_valid, wv);
    atomicAdd(&d.cnt->tracklet_hits, (unsigned long long)wh);
  }
}

// (e4) every hit of a valid tracklet receives max(weight) (O5 "Result").  One warp per seed: lanes take
// consecutive rows, so the row_hit reads are coalesced and 32 atomics are in flight per warp.
__global__ void __launch_bounds__(128) k_tracklet_weights(Dev d) {
  const int lane = threadIdx.x & 31;
  const int n_work = d.cnt->n_work, n_warps = (gridDim.x * 128) >> 5;
  for (int w = (blockIdx.x * 128 + threadIdx.x) >> 5; w < n_work; w += n_warps) {
    const int t = d.work_t[w];
    const int4 ti = reinterpret_cast<const int4*>(d.tl_ints)[t];
    if (!ti.x) continue;
    const unsigned long long W = d.tl_W[t];
    const int32_t* rh = d.row_hit + (size_t)w * d.n_rows;
    for (int r = ti.y + lane; r <= ti.z; r += 32) {
      const int h = rh[r];
      if (h >= 0) atomicMax(&d.hit_weight[h], W);
    }
  }
}

#ifndef W_GRID
#define W_GRID 8  // CTAs per SM of k_tracklet_weights: the L2 atomic units saturate with 32 warps per SM (16: +0.07 ms)
#endif
#ifndef E2_GRID
#define E2_GRID E2_BLOCKS
#endif
#ifndef E3_GRID
#define E3_GRID E3_BLOCKS
#endif
void launch_tracklets(const Dev& d, Launch& L) {
  if (d.n <= 0 || d.max_tracklets <= 0) return;
  const int T = d.max_tracklets;
  k_seed_flag<<<(T + 255) / 256, 256, 0, L.st>>>(d);
  L.count++;
  launch_scan_i32(d.seed_w, &d.cnt->n_start, T, d.scan_tmp, L);
  k_seed_compact<<<(T + 255) / 256, 256, 0, L.st>>>(d);
  KTIMED(L, TPCCA_K_TL_E1, (k_tl_e1<<<d.n_sm * E1_BLOCKS, E_THREADS, 0, L.st>>>(d)));
  launch_order_desc(d, 1, d.e_key, &d.cnt->n_work, T, d.e_order, L);
  KTIMED(L, TPCCA_K_TL_E2, (k_tl_e2<<<d.n_sm * E2_GRID, E_THREADS, 0, L.st>>>(d)));
  launch_order_desc(d, 2, d.e_key + T, &d.cnt->n_work, T, d.e_order + T, L);
  KTIMED(L, TPCCA_K_TL_E3A, (k_tl_e3a<<<d.n_sm * E3_GRID, E_THREADS, 0, L.st>>>(d)));
  launch_order_desc(d, 3, d.e_key + 2 * (size_t)T, &d.cnt->n_work, T, d.e_order + 2 * (size_t)T, L);
  KTIMED(L, TPCCA_K_TL_E3B, (k_tl_e3b<<<d.n_sm * E3B_BLOCKS, E_THREADS, 0, L.st>>>(d)));
  KTIMED(L, TPCCA_K_WEIGHTS, (k_tracklet_weights<<<d.n_sm * W_GRID, 128, 0, L.st>>>(d)));
  L.count += 6;
}
