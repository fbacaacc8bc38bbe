// tpcca_oracle.cpp -- TEST INFRASTRUCTURE, NOT PRODUCT CODE.
//
// Plain, single-threaded CPU oracle for the per-sector cellular-automaton track finder and
// Kalman fit of arXiv 1811.11481 (PAPER.md:49-51 phase 1; :65-68 outward then inward through
// the seed with outlier rejection; :71 three-pass refit; :98/:104 no vertex constraint, window
// centred on the hit; :121 fp32, z kept relative).  It follows the algorithm step by step in
// the order of DESIGN.md section "Arithmetic" (steps O1-O7) and shares no code with the CUDA path.
// Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may
// load it.  Build: g++ -O2 -ffp-contract=off (no fast-math): every decision is fp32; the compiler never contracts a
// multiply-add on its own -- the fused operations are exactly the fma() calls DESIGN.md section 3 states (std::fma is
// correctly rounded on every platform, with or without hardware support).
//
// Pins (tests/test_oracle_pins.py): brute-force all-triplet search (P1), noiseless helix (P2),
// mutual links (P3), exclusive assignment (P4), permutation invariance (P5), transport closed
// form (P6), straight-line least squares (P7), pulls (P8), -O0 == -O2 (P10).
// Merger and final fit O8-O10: tests/test_merge_pins.py; z / time estimate O11: tests/test_time_pins.py; looper legs and
// cluster tags O12-O13: tests/test_looper_pins.py (float64 closed-form helices
// over all sectors, the angle polynomial against arctan2, every term of the pair score, 54 one-line mutants all fail a pin).
// Parity unpinned: the numeric defaults of DESIGN.md Tables A, B and D (cuts, windows, cov0) -- the paper
// prints no value for them.
#include <algorithm>
#include <cmath>
#include <cstdint>
#include <cstring>
#include <vector>

namespace {

struct Params {  // mirrors DESIGN.md Table A; filled field by field from Python
  float sigma_y, sigma_z;
  float nbr_dydx, nbr_dzdx, nbr_margin_y, nbr_margin_z, triplet_cut;
  float cov0[5];
  float pick_cut, reject_cut;
  int32_t max_gap;
  float edge_margin, max_sinphi;
  int32_t min_seed_hits, min_tracklet_hits, min_track_hits;
  float qual_scale;
  float tan_half_angle;
};

struct Cl { float x, y, z; int32_t row; };

struct TrackRec {  // 128 bytes, same field order as the product's record (declared independently)
  int32_t sector, first_row, last_row, n_hits;
  float x, y, z, sinphi, dzds, qpt;
  float cov[15];
  float chi2;
  int32_t ndf;
  int32_t pad[5];
};

struct KF {
  float x;
  float p[5];   // y, z~ (relative to z_ref), sin(phi), dz/ds, q/pT
  float C[15];  // lower triangle, row major: C[i*(i+1)/2+j], i>=j
  float chi2;
};

inline float fma32(float a, float b, float c) { return std::fma(a, b, c); }  // one rounding: the "fma(a,b,c)" of DESIGN.md

inline uint32_t ordf(float f) {  // monotone float -> uint map
  uint32_t b;
  std::memcpy(&b, &f, 4);
  return (b & 0x80000000u) ? ~b : (b | 0x80000000u);
}

inline int tri(int i, int j) { return i >= j ? i * (i + 1) / 2 + j : j * (j + 1) / 2 + i; }

// ---- O5 model: transport x -> xnew (DESIGN.md section 3 "Transport") ----
// The step is written as the textbook extended-Kalman prediction: move the state along the helix, fill the dense
// 5x5 Jacobian F = d(y, z~, s, t, q)' / d(y, z~, s, t, q), then C <- F C F^T by the two matrix products of the
// definition.  DESIGN.md section 3 fixes the summation order: every entry starts from the unit-diagonal term and
// accumulates the remaining terms in increasing k by fma(F_ik, C_kj, acc); a term whose Jacobian entry is structurally
// zero (see `nz`) is left out rather than added as 0 * c.
bool transport(KF& k, float xnew, float kq, float max_sinphi) {
  const float dx = xnew - k.x;
  if (dx == 0.0f) return true;  // identity (first step of E3 and of every refit pass)
  const float s0 = k.p[2], tl = k.p[3];
  const float curv = k.p[4] * kq;  // d sin(phi) / dx
  const float s1 = fma32(dx, curv, s0);
  if (!(std::fabs(s0) <= max_sinphi)) return false;
  if (!(std::fabs(s1) <= max_sinphi)) return false;
  // helix step: chord direction f = tan of the mean angle, chord length L (signed like dx), arc = L * asin(u)/u
  const float cos0 = std::sqrt(fma32(-s0, s0, 1.0f));
  const float cos1 = std::sqrt(fma32(-s1, s1, 1.0f));
  const float csum = cos0 + cos1;
  // the three quotients by cos0, cos1 and their sum share ONE division: inv = 1 / (cos0 cos1 csum)
  const float c01 = cos0 * cos1;
  const float inv = 1.0f / (c01 * csum);
  const float icsum = c01 * inv, icos0 = (cos1 * csum) * inv, icos1 = (cos0 * csum) * inv;
  const float f = (s0 + s1) * icsum;
  const float dy = dx * f;
  float L = std::sqrt(fma32(dx, dx, dy * dy));
  if (dx < 0.0f) L = -L;
  const float u = (0.5f * curv) * L;
  const float u2 = u * u;
  const float g = fma32(u2, fma32(u2, 0.075f, 0.16666667f), 1.0f);  // asin(u)/u = 1 + u^2/6 + 3u^4/40 + ...
  const float arc = L * g;
  // Jacobian (d g neglected): d f / d s0 and d f / d s1, then the chain rule through s1 = s0 + dx * kq * q
  const float df_ds0 = fma32(f * s0, icos0, 1.0f) * icsum;
  const float df_ds1 = fma32(f * s1, icos1, 1.0f) * icsum;
  const float ds1_dq = dx * kq;
  const float df_ds = df_ds0 + df_ds1;
  const float darc_df = (tl * g) * ((dx * dy) / L);  // d(z~)/df = t * g * dL/df, dL/df = dx*dy/L
  float F[5][5];
  bool nz[5][5];
  for (int i = 0; i < 5; i++)
    for (int j = 0; j < 5; j++) { F[i][j] = (i == j) ? 1.0f : 0.0f; nz[i][j] = (i == j); }
  F[0][2] = dx * df_ds;               nz[0][2] = true;
  F[0][4] = (dx * df_ds1) * ds1_dq;   nz[0][4] = true;
  F[1][2] = darc_df * df_ds;          nz[1][2] = true;
  F[1][3] = arc;                      nz[1][3] = true;
  F[1][4] = (darc_df * df_ds1) * ds1_dq; nz[1][4] = true;
  F[2][4] = ds1_dq;                   nz[2][4] = true;
  // state
  k.p[0] = k.p[0] + dy;
  k.p[1] = fma32(tl, arc, k.p[1]);
  k.p[2] = s1;
  k.x = xnew;
  // covariance: full symmetric C, M = F C, C' = M F^T (lower triangle kept)
  float Cf[5][5], M[5][5];
  for (int i = 0; i < 5; i++)
    for (int j = 0; j < 5; j++) Cf[i][j] = k.C[tri(i, j)];
  for (int i = 0; i < 5; i++)
    for (int j = 0; j < 5; j++) {
      float acc = 0.0f;
      bool first = true;
      for (int l = 0; l < 5; l++) {
        if (!nz[i][l]) continue;
        acc = first ? Cf[l][j] : fma32(F[i][l], Cf[l][j], acc);  // first non-zero of row i is F_ii = 1
        first = false;
      }
      M[i][j] = acc;
    }
  for (int i = 0; i < 5; i++)
    for (int j = 0; j <= i; j++) {
      float acc = 0.0f;
      bool first = true;
      for (int l = 0; l < 5; l++) {
        if (!nz[j][l]) continue;
        acc = first ? M[i][l] : fma32(F[j][l], M[i][l], acc);
        first = false;
      }
      k.C[tri(i, j)] = acc;
    }
  return true;
}

// ---- O5 model: scalar measurement update of component i (0: y, 1: z~) ----
void update1(KF& k, int i, float m, float v) {
  float ci[5];
  for (int j = 0; j < 5; j++) ci[j] = k.C[tri(j, i)];
  const float r = m - k.p[i];
  const float S = ci[i] + v;
  const float w = 1.0f / S;
  float K[5];
  for (int j = 0; j < 5; j++) K[j] = ci[j] * w;
  for (int j = 0; j < 5; j++) k.p[j] = fma32(K[j], r, k.p[j]);
  for (int j = 0; j < 5; j++)
    for (int l = 0; l <= j; l++) k.C[tri(j, l)] = fma32(-K[j], ci[l], k.C[tri(j, l)]);
  k.chi2 = fma32(r * r, w, k.chi2);
}

void update(KF& k, float ym, float zm_rel, float sy2, float sz2) {
  update1(k, 0, ym, sy2);
  update1(k, 1, zm_rel, sz2);
}

void reset_cov(KF& k, const Params& P) {
  for (int i = 0; i < 15; i++) k.C[i] = 0.0f;
  for (int i = 0; i < 5; i++) k.C[tri(i, i)] = P.cov0[i];
  k.chi2 = 0.0f;
}

struct Tracklet {
  int32_t sector, start_hit;  // start_hit: input index
  int32_t valid, first_row, last_row, n_hits;
  float x, p[5], C[15], chi2, z_ref;
  uint64_t W;
};

struct Result {
  int64_t n = 0;
  int32_t n_sectors = 0, n_rows = 0;
  std::vector<int32_t> link_up_raw, link_down_raw, link_up, link_down;  // input-index space
  std::vector<int32_t> start_hits;                                       // input indices, canonical order
  std::vector<Tracklet> tracklets;
  std::vector<int32_t> row_hit;  // n_tracklets * n_rows, input indices or -1
  std::vector<int32_t> assignment;
  std::vector<TrackRec> tracks;
  std::vector<int32_t> track_tracklet;
  // kept for the merger (O8-O10)
  std::vector<std::vector<int32_t>> track_hits;  // per sector track: input indices, increasing row
  std::vector<KF> outer;                         // state at the outermost hit after the outward refit pass (z~ relative)
  std::vector<float> outer_zref;
  std::vector<uint8_t> shared;                   // per cluster: also collected by the tracklet of another accepted track
  // merger output
  std::vector<TrackRec> merged;
  std::vector<int32_t> track_merged;             // sector track -> merged track
  std::vector<int32_t> link_next;                // sector track -> sector track it continues into, or -1
  // looper legs and cluster tags (O12, O13)
  std::vector<int32_t> leg_partner;              // merged track -> merged track joined at the outer turning point, or -1
  std::vector<int32_t> leg_partner_in;           // merged track -> merged track joined through the inner region, or -1
  std::vector<uint8_t> leg_first;                // merged track: 1 = first (or only) leg, 0 = additional leg
  std::vector<uint8_t> cluster_tags;             // per cluster: TAG_* bits
  std::vector<TrackRec> leg_fits;                // O14: one fit per pair of legs joined at a turning point
};

struct Sector {
  const Cl* cl;                              // all clusters (input order)
  std::vector<std::vector<int32_t>> rows;    // per row: input indices sorted by key (z, y, idx)
};

struct Ctx {
  const Cl* cl;
  const float* row_x;
  int n_rows;
  Params P;
  float kq, sy2, sz2, inv_sy2, inv_sz2;
  bool brute;
};

inline bool key_less(const Cl* cl, int32_t a, int32_t b) {  // same-row key: (ord z, ord y, input index)
  const uint32_t za = ordf(cl[a].z), zb = ordf(cl[b].z);
  if (za != zb) return za < zb;
  const uint32_t ya = ordf(cl[a].y), yb = ordf(cl[b].y);
  if (ya != yb) return ya < yb;
  return a < b;
}

// Candidates of a row with z in [zlo, zhi] (a superset is fine; exact predicates are applied by the caller).
inline void z_range(const Ctx& c, const std::vector<int32_t>& row, double zlo, double zhi, size_t& b, size_t& e) {
  if (c.brute) { b = 0; e = row.size(); return; }
  const Cl* cl = c.cl;
  b = std::lower_bound(row.begin(), row.end(), zlo, [cl](int32_t i, double z) { return (double)cl[i].z < z; }) - row.begin();
  e = std::upper_bound(row.begin(), row.end(), zhi, [cl](double z, int32_t i) { return z < (double)cl[i].z; }) - row.begin();
  if (!(zlo <= zhi)) { b = 0; e = 0; }  // NaN window: nothing can pass the exact predicate
}

// ---- O2 neighbours finder for one sector ----
void find_neighbours(const Ctx& c, const Sector& S, std::vector<int32_t>& up, std::vector<int32_t>& down) {
  const int R = c.n_rows;
  const Cl* cl = c.cl;
  const Params& P = c.P;
  std::vector<int32_t> U, D;
  for (int r = 0; r < R; r++) {
    int ru = -1, rd = -1;
    if (r + 1 < R && !S.rows[r + 1].empty()) ru = r + 1;
    else if (r + 2 < R && !S.rows[r + 2].empty()) ru = r + 2;
    if (r - 1 >= 0 && !S.rows[r - 1].empty()) rd = r - 1;
    else if (r - 2 >= 0 && !S.rows[r - 2].empty()) rd = r - 2;
    if (ru < 0 || rd < 0) continue;  // links stay -1
    const float dxu = c.row_x[ru] - c.row_x[r];
    const float dxd = c.row_x[r] - c.row_x[rd];
    const float t = dxd / (dxu + dxd);
    const float wyu = fma32(dxu, P.nbr_dydx, P.nbr_margin_y);
    const float wzu = fma32(dxu, P.nbr_dzdx, P.nbr_margin_z);
    const float wyd = fma32(dxd, P.nbr_dydx, P.nbr_margin_y);
    const float wzd = fma32(dxd, P.nbr_dzdx, P.nbr_margin_z);
    for (int32_t h : S.rows[r]) {
      const float y0 = cl[h].y, z0 = cl[h].z;
      U.clear(); D.clear();
      size_t b, e;
      z_range(c, S.rows[ru], (double)z0 - wzu - 0.01, (double)z0 + wzu + 0.01, b, e);
      for (size_t i = b; i < e; i++) {
        const int32_t u = S.rows[ru][i];
        if (std::fabs(cl[u].y - y0) <= wyu && std::fabs(cl[u].z - z0) <= wzu) U.push_back(u);
      }
      z_range(c, S.rows[rd], (double)z0 - wzd - 0.01, (double)z0 + wzd + 0.01, b, e);
      for (size_t i = b; i < e; i++) {
        const int32_t d = S.rows[rd][i];
        if (std::fabs(cl[d].y - y0) <= wyd && std::fabs(cl[d].z - z0) <= wzd) D.push_back(d);
      }
      int32_t bu = -1, bd = -1;
      float bc = 0.0f;
      for (int32_t u : U)
        for (int32_t d : D) {
          const float yu = cl[u].y, zu = cl[u].z, yd = cl[d].y, zd = cl[d].z;
          const float ey = y0 - fma32(t, yu - yd, yd);
          const float ez = z0 - fma32(t, zu - zd, zd);
          const float cost = fma32(ez * ez, c.inv_sz2, (ey * ey) * c.inv_sy2);
          if (!(cost <= P.triplet_cut)) continue;
          bool better;
          if (bu < 0) better = true;
          else if (cost != bc) better = cost < bc;
          else if (u != bu) better = key_less(cl, u, bu);
          else better = key_less(cl, d, bd);
          if (better) { bu = u; bd = d; bc = cost; }
        }
      up[h] = bu;
      down[h] = bd;
    }
  }
}

// Best pick-up candidate in a row for the predicted state (O5 "search"); returns input index or -1.
int32_t search_row(const Ctx& c, const std::vector<int32_t>& row, const KF& k, float z_ref, float cut) {
  if (row.empty()) return -1;
  const Cl* cl = c.cl;
  const float vy = k.C[0] + c.sy2, vz = k.C[2] + c.sz2;
  const float iy = 1.0f / vy, iz = 1.0f / vz;
  const float wy = std::sqrt(cut * vy), wz = std::sqrt(cut * vz);
  const double zc = (double)z_ref + (double)k.p[1];
  size_t b, e;
  const double m = 0.01 + 1e-6 * std::fabs(zc);
  z_range(c, row, zc - (double)wz - m, zc + (double)wz + m, b, e);
  int32_t best = -1;
  float bd = 0.0f;
  for (size_t i = b; i < e; i++) {
    const int32_t h = row[i];
    const float dy = cl[h].y - k.p[0];
    const float dz = (cl[h].z - z_ref) - k.p[1];
    if (!(std::fabs(dy) <= wy) || !(std::fabs(dz) <= wz)) continue;
    const float d = fma32(dz * dz, iz, (dy * dy) * iy);
    if (!(d <= cut)) continue;
    bool better;
    if (best < 0) better = true;
    else if (d != bd) better = d < bd;
    else better = key_less(cl, h, best);
    if (better) { best = h; bd = d; }
  }
  return best;
}

inline float hit_dist(const Ctx& c, const KF& k, const Cl& h, float z_ref) {
  const float iy = 1.0f / (k.C[0] + c.sy2), iz = 1.0f / (k.C[2] + c.sz2);
  const float dy = h.y - k.p[0];
  const float dz = (h.z - z_ref) - k.p[1];
  return fma32(dz * dz, iz, (dy * dy) * iy);
}

// ---- O5 tracklet construction for one start hit ----
void build_tracklet(const Ctx& c, const Sector& S, const std::vector<int32_t>& link_up, int32_t h0, Tracklet& T,
                    int32_t* row_hit /* n_rows, preset to -1 */) {
  const Params& P = c.P;
  const Cl* cl = c.cl;
  const int R = c.n_rows;
  T.valid = 0; T.first_row = T.last_row = -1; T.n_hits = 0; T.W = 0; T.chi2 = 0; T.x = 0;
  for (int i = 0; i < 5; i++) T.p[i] = 0;
  for (int i = 0; i < 15; i++) T.C[i] = 0;
  const float z_ref = cl[h0].z;
  T.z_ref = z_ref;
  // E1: seed fit outward along the links
  const int32_t h1 = link_up[h0];
  KF k;
  {
    const float dx = cl[h1].x - cl[h0].x, dy = cl[h1].y - cl[h0].y, dz = cl[h1].z - cl[h0].z;
    const float ds = std::sqrt(fma32(dx, dx, dy * dy));
    k.x = cl[h0].x;
    k.p[0] = cl[h0].y; k.p[1] = 0.0f; k.p[2] = dy / ds; k.p[3] = dz / ds; k.p[4] = 0.0f;
    reset_cov(k, P);
  }
  update(k, cl[h0].y, cl[h0].z - z_ref, c.sy2, c.sz2);
  row_hit[cl[h0].row] = h0;
  int n_chain = 1, last_row = cl[h0].row;
  for (int32_t h = h1; h >= 0; h = link_up[h]) {
    if (!transport(k, cl[h].x, c.kq, P.max_sinphi)) return;  // void
    update(k, cl[h].y, cl[h].z - z_ref, c.sy2, c.sz2);
    row_hit[cl[h].row] = h;
    last_row = cl[h].row;
    n_chain++;
  }
  if (n_chain < P.min_seed_hits) return;  // void
  const int r_low = cl[h0].row;
  // E2: outward extrapolation, one best cluster per row
  KF snap = k;  // state at the outermost hit
  int top_row = last_row, gap = 0;
  for (int r = last_row + 1; r < R; r++) {
    if (!transport(k, c.row_x[r], c.kq, P.max_sinphi)) break;
    if (std::fabs(k.p[0]) > fma32(c.row_x[r], P.tan_half_angle, P.edge_margin)) break;
    const int32_t hb = search_row(c, S.rows[r], k, z_ref, P.pick_cut);
    if (hb >= 0) {
      update(k, cl[hb].y, cl[hb].z - z_ref, c.sy2, c.sz2);
      row_hit[r] = hb; gap = 0; snap = k; top_row = r;
    } else {
      gap++;
      if (gap > P.max_gap) break;
    }
  }
  // E3: inward pass through the seed with outlier rejection, then pick-up below it
  k = snap;
  reset_cov(k, P);
  KF inner = k;
  int inner_row = -1;
  gap = 0;
  int r = top_row;
  for (; r >= 0; r--) {
    if (!transport(k, c.row_x[r], c.kq, P.max_sinphi)) break;
    if (std::fabs(k.p[0]) > fma32(c.row_x[r], P.tan_half_angle, P.edge_margin)) break;
    bool hit = false;
    if (row_hit[r] >= 0) {
      const Cl& hc = cl[row_hit[r]];
      const float d = hit_dist(c, k, hc, z_ref);
      if (d <= P.reject_cut) { update(k, hc.y, hc.z - z_ref, c.sy2, c.sz2); hit = true; }
      else row_hit[r] = -1;
    } else {
      const int32_t hb = search_row(c, S.rows[r], k, z_ref, P.pick_cut);
      if (hb >= 0) { update(k, cl[hb].y, cl[hb].z - z_ref, c.sy2, c.sz2); row_hit[r] = hb; hit = true; }
    }
    if (hit) { gap = 0; inner = k; inner_row = r; }
    else { gap++; if (r < r_low && gap > P.max_gap) { r--; break; } }
  }
  for (int rr = r; rr >= 0; rr--) row_hit[rr] = -1;  // rows the pass never reached (or stopped on)
  if (inner_row < 0) return;
  int n_hits = 0, first = -1, last = -1;
  for (int rr = 0; rr < R; rr++)
    if (row_hit[rr] >= 0) { n_hits++; if (first < 0) first = rr; last = rr; }
  if (n_hits < P.min_tracklet_hits) return;
  T.valid = 1; T.first_row = first; T.last_row = last; T.n_hits = n_hits;
  T.x = inner.x; T.chi2 = inner.chi2;
  for (int i = 0; i < 5; i++) T.p[i] = inner.p[i];
  for (int i = 0; i < 15; i++) T.C[i] = inner.C[i];
}

inline uint64_t pack_weight(const Params& P, int n_hits, float chi2, uint32_t tid) {
  float qf = (P.qual_scale * chi2) / (float)(2 * n_hits);
  qf = std::fmin(65535.0f, qf);
  qf = std::fmax(0.0f, qf);
  const int qi = (int)qf;
  const uint32_t qual = (uint32_t)(65535 - qi);
  return ((uint64_t)(uint32_t)n_hits << 48) | ((uint64_t)qual << 32) | (uint64_t)(0xFFFFFFFFu - tid);
}

// ---- O7 refit: inward, outward, inward over the track's hits ----
// hits: input indices in increasing row order.  Returns false if a transport failed.
bool refit(const Ctx& c, const std::vector<int32_t>& hits, float q0, KF& k, float& z_ref, KF* outer = nullptr) {
  const Cl* cl = c.cl;
  const int n = (int)hits.size();
  const Cl& hN = cl[hits[n - 1]];
  const Cl& hM = cl[hits[n - 2]];
  z_ref = hN.z;
  const float dx = hN.x - hM.x, dy = hN.y - hM.y, dz = hN.z - hM.z;
  const float ds = std::sqrt(fma32(dx, dx, dy * dy));
  k.x = hN.x;
  k.p[0] = hN.y; k.p[1] = 0.0f; k.p[2] = dy / ds; k.p[3] = dz / ds; k.p[4] = q0;
  for (int pass = 0; pass < 3; pass++) {
    reset_cov(k, c.P);
    for (int j = 0; j < n; j++) {
      const Cl& h = cl[hits[(pass == 1) ? j : n - 1 - j]];
      if (!transport(k, h.x, c.kq, c.P.max_sinphi)) return false;
      update(k, h.y, h.z - z_ref, c.sy2, c.sz2);
    }
    if (pass == 1 && outer) *outer = k;  // end of the outward pass: the state at the outermost hit (O8)
  }
  return true;
}

Ctx make_ctx(const Cl* cl, const float* row_x, int n_rows, const Params& P, float bz, bool brute) {
  Ctx c;
  c.cl = cl; c.row_x = row_x; c.n_rows = n_rows; c.P = P; c.brute = brute;
  c.kq = -((0.000299792458f * 10.0f) * bz);
  c.sy2 = P.sigma_y * P.sigma_y;
  c.sz2 = P.sigma_z * P.sigma_z;
  c.inv_sy2 = 1.0f / c.sy2;
  c.inv_sz2 = 1.0f / c.sz2;
  return c;
}

// ---- O8-O10: sector-segment merger and final fit (PAPER.md:51 second phase; :69-71) ----
struct MergeParams {
  float merge_chi2_cut, merge_dz_max, merge_edge_dist;
  int32_t merge_row_back, merge_row_fwd;
  float fit_reject_cut, shared_err_scale;
  int32_t ring;  // sectors per z side that close the ring (18), 0: no neighbours
};

// Change of the sector frame by sgn * 20 degrees (sgn = +1: into the next sector).  cos / sin of the sector angle come
// from tan(10 deg) by the double-angle formulas (no libm).  false: |sin(phi)| leaves [-max_sinphi, max_sinphi].
bool rotate_frame(KF& k, float ca, float ss, float kq, float max_sinphi) {
  const float s = k.p[2];
  if (!(std::fabs(s) <= max_sinphi)) return false;
  const float cphi = std::sqrt(fma32(-s, s, 1.0f));
  const float s1 = fma32(s, ca, -(cphi * ss));
  if (!(std::fabs(s1) <= max_sinphi)) return false;
  const float c1 = std::sqrt(fma32(-s1, s1, 1.0f));
  // Jacobian of "state on the plane x = const" -> "state on the plane x' = const through the same point":
  // a shift of y moves the point off the new plane; sliding back along the track gives dy'/dy = cos(phi)/cos(phi'),
  // dz'/dy = -t sin(a)/cos(phi'), d sin(phi')/dy = -(q kq) sin(a) (the slide changes sin(phi) by the curvature);
  // d sin(phi')/d sin(phi) = cos(phi')/cos(phi).  F = diag(ry, 1, rr, 1, 1) + rz at (1,0) + rs at (2,0).
  const float rr = c1 / cphi;
  const float ry = cphi / c1;
  const float rz = -((k.p[3] * ss) / c1);
  const float rs = -((k.p[4] * kq) * ss);
  const float x = k.x, y = k.p[0];
  k.x = fma32(y, ss, x * ca);
  k.p[0] = fma32(y, ca, -(x * ss));
  k.p[2] = s1;
  float Cf[5][5], Mx[5][5];
  for (int i = 0; i < 5; i++)
    for (int j = 0; j < 5; j++) Cf[i][j] = k.C[tri(i, j)];
  for (int j = 0; j < 5; j++) {  // M = F C
    Mx[0][j] = ry * Cf[0][j];
    Mx[1][j] = fma32(rz, Cf[0][j], Cf[1][j]);
    Mx[2][j] = fma32(rs, Cf[0][j], rr * Cf[2][j]);
    Mx[3][j] = Cf[3][j];
    Mx[4][j] = Cf[4][j];
  }
  for (int i = 0; i < 5; i++) {  // C' = M F^T, lower triangle
    k.C[tri(i, 0)] = Mx[i][0] * ry;
    if (i >= 1) k.C[tri(i, 1)] = fma32(rz, Mx[i][0], Mx[i][1]);
    if (i >= 2) k.C[tri(i, 2)] = fma32(rs, Mx[i][0], Mx[i][2] * rr);
    if (i >= 3) k.C[tri(i, 3)] = Mx[i][3];
    if (i >= 4) k.C[tri(i, 4)] = Mx[i][4];
  }
  return true;
}

inline int ring_neighbour(int sector, int side, int ring) {  // side = +1 / -1; -1 if there is none
  if (ring <= 0) return -1;
  const int base = (sector / ring) * ring, l = sector - base;
  return base + (l + side + ring) % ring;
}

void merge_tracks(Result* R, const Ctx& c, const MergeParams& M) {
  const Cl* cl = c.cl;
  const Params& P = c.P;
  const int nt = (int)R->tracks.size();
  const float th = P.tan_half_angle;
  const float den = fma32(th, th, 1.0f);
  const float ca = fma32(-th, th, 1.0f) / den, sa = (2.0f * th) / den;  // cos, sin of the sector angle
  // O9: best partner of every outer end, best partner of every inner end
  std::vector<int32_t> best_out(nt, -1), best_in(nt, -1);
  std::vector<float> chi_out(nt, 0.0f), chi_in(nt, 0.0f);
  std::vector<std::vector<int32_t>> by_sector(R->n_sectors);  // track ids per sector, increasing
  for (int t = 0; t < nt; t++) by_sector[R->tracks[t].sector].push_back(t);
  for (int a = 0; a < nt; a++) {
    const TrackRec& A = R->tracks[a];
    if (A.ndf < 0) continue;
    const KF& oa = R->outer[a];
    const float za = oa.p[1] + R->outer_zref[a];
    const int side = oa.p[0] > 0.0f ? 1 : -1;
    if (!(std::fabs(oa.p[0]) >= fma32(oa.x, th, -M.merge_edge_dist))) continue;
    const int sb = ring_neighbour(A.sector, side, M.ring);
    if (sb < 0 || sb >= R->n_sectors) continue;
    for (int b : by_sector[sb]) {
      const TrackRec& B = R->tracks[b];
      if (B.ndf < 0) continue;
      const int dr = B.first_row - A.last_row;
      if (dr < -M.merge_row_back || dr > M.merge_row_fwd) continue;
      if (!(std::fabs(B.z - za) <= M.merge_dz_max)) continue;
      KF k = oa;
      k.p[1] = 0.0f;  // z relative to the outer end of A
      if (!rotate_frame(k, ca, (float)side * sa, c.kq, P.max_sinphi)) continue;
      if (!transport(k, B.x, c.kq, P.max_sinphi)) continue;
      const float pb[5] = {B.y, B.z - za, B.sinphi, B.dzds, B.qpt};
      float chi = 0.0f;
      for (int i = 0; i < 5; i++) {
        const float d = k.p[i] - pb[i];
        const float term = (d * d) / (k.C[tri(i, i)] + B.cov[tri(i, i)]);
        chi = (i == 0) ? term : chi + term;
      }
      if (!(chi <= M.merge_chi2_cut)) continue;
      if (best_out[a] < 0 || chi < chi_out[a]) { best_out[a] = b; chi_out[a] = chi; }       // equal chi2: lower id of B stays
      if (best_in[b] < 0 || chi < chi_in[b]) { best_in[b] = a; chi_in[b] = chi; }           // equal chi2: lower id of A stays
    }
  }
  R->link_next.assign(nt, -1);
  std::vector<int32_t> prev(nt, -1);
  for (int a = 0; a < nt; a++) {
    const int b = best_out[a];
    if (b >= 0 && best_in[b] == a) { R->link_next[a] = b; prev[b] = a; }
  }
  // O10: chains from the heads in id order, final three-pass fit with rejection
  R->track_merged.assign(nt, -1);
  R->merged.clear();
  for (int head = 0; head < nt; head++) {
    if (prev[head] >= 0) continue;
    const int32_t mid = (int32_t)R->merged.size();
    std::vector<int32_t> hits, hsec;  // inner -> outer
    int n_seg = 0, last = head;
    for (int t = head; t >= 0; t = R->link_next[t]) {
      R->track_merged[t] = mid;
      for (int32_t h : R->track_hits[t]) { hits.push_back(h); hsec.push_back(R->tracks[t].sector); }
      n_seg++; last = t;
    }
    const int n = (int)hits.size();
    TrackRec tr;
    std::memset(&tr, 0, sizeof(tr));
    tr.sector = R->tracks[head].sector; tr.first_row = cl[hits.front()].row; tr.last_row = cl[hits.back()].row;
    tr.n_hits = n;
    const Cl& hN = cl[hits[n - 1]];
    const Cl& hM = cl[hits[n - 2]];  // same segment: a sector track has >= 2 hits
    const float z_ref = hN.z;
    KF k;
    {
      const float dx = hN.x - hM.x, dy = hN.y - hM.y, dz = hN.z - hM.z;
      const float ds = std::sqrt(fma32(dx, dx, dy * dy));
      k.x = hN.x;
      k.p[0] = hN.y; k.p[1] = 0.0f; k.p[2] = dy / ds; k.p[3] = dz / ds; k.p[4] = R->tracks[last].qpt;
    }
    bool ok = true;
    int n_used = 0, n_shared = 0;
    int cur_sec = hsec[n - 1];
    for (int pass = 0; pass < 3 && ok; pass++) {
      reset_cov(k, P);
      n_used = 0; n_shared = 0;
      for (int j = 0; j < n && ok; j++) {
        const int idx = (pass == 1) ? j : n - 1 - j;
        const Cl& h = cl[hits[idx]];
        if (hsec[idx] != cur_sec) {  // adjacent sectors by construction of the chain
          const int sgn = (ring_neighbour(cur_sec, +1, M.ring) == hsec[idx]) ? 1 : -1;
          if (!rotate_frame(k, ca, (float)sgn * sa, c.kq, P.max_sinphi)) { ok = false; break; }
          cur_sec = hsec[idx];
        }
        if (!transport(k, h.x, c.kq, P.max_sinphi)) { ok = false; break; }
        const bool sh = R->shared[hits[idx]] != 0;
        const float ey = sh ? P.sigma_y * M.shared_err_scale : P.sigma_y;
        const float ez = sh ? P.sigma_z * M.shared_err_scale : P.sigma_z;
        const float vy = ey * ey, vz = ez * ez;
        n_shared += sh ? 1 : 0;
        const float iy = 1.0f / (k.C[0] + vy), iz = 1.0f / (k.C[2] + vz);
        const float dy = h.y - k.p[0];
        const float dz = (h.z - z_ref) - k.p[1];
        const float d = fma32(dz * dz, iz, (dy * dy) * iy);
        if (!(d <= M.fit_reject_cut)) continue;  // outlier for this pass
        update(k, h.y, h.z - z_ref, vy, vz);
        n_used++;
      }
    }
    if (ok) {
      tr.x = k.x; tr.y = k.p[0]; tr.z = k.p[1] + z_ref; tr.sinphi = k.p[2]; tr.dzds = k.p[3]; tr.qpt = k.p[4];
      for (int i = 0; i < 15; i++) tr.cov[i] = k.C[i];
      tr.chi2 = k.chi2;
      tr.ndf = 2 * n_used - 5;
    } else {  // a rotation or transport left |sin(phi)| <= max_sinphi: keep the innermost segment's own fit, flagged
      const TrackRec& H = R->tracks[head];
      tr.x = H.x; tr.y = H.y; tr.z = H.z; tr.sinphi = H.sinphi; tr.dzds = H.dzds; tr.qpt = H.qpt;
      for (int i = 0; i < 15; i++) tr.cov[i] = H.cov[i];
      tr.chi2 = H.chi2;
      tr.ndf = -1;
    }
    tr.pad[0] = n_seg; tr.pad[1] = R->tracks[last].sector; tr.pad[2] = ok ? n - n_used : -1; tr.pad[3] = n_shared;
    tr.pad[4] = head;
    R->merged.push_back(tr);
  }
}

// ---- O11: z / time estimate of a track in a time frame ----
// Plain definition in double precision from the fp32 track record: the point of closest approach of the helix to the
// beam line (x = y = 0 in every sector frame), its z, and the shift that brings the track's clusters inside the drift volume.
struct TimeRec { float z_dca, z_shift, t0_us, dca_xy; };

TimeRec time_estimate(const TrackRec& T, double kq, double zmin_hits, double zmax_hits, int side, double vdrift, double z_max) {
  const double x = T.x, y = T.y, s = T.sinphi, c = std::sqrt(1.0 - s * s), k = (double)T.qpt * kq;
  double ds, dca;  // path length from the state to the closest approach (negative: behind), signed distance there
  if (std::fabs(k) < 1e-12) {
    ds = -(c * x + s * y);
    dca = y * c - x * s;
  } else {
    const double R = 1.0 / std::fabs(k), sg = k > 0 ? 1.0 : -1.0;
    const double xc = x - s / k, yc = y + c / k;          // circle centre: left of the direction by 1/k
    const double Rc = std::sqrt(xc * xc + yc * yc);
    // turning angle from the state to the point of the circle nearest to the origin (on the line origin -> centre)
    const double dphi = std::atan2(-sg * (c * x + s * y), R - sg * (s * x - c * y));
    ds = dphi / k;
    dca = sg * (Rc - R);  // same sign convention as the straight line: the state's offset along its left normal
  }
  TimeRec o;
  const double zd = (double)T.z + (double)T.dzds * ds;
  // shift so that the clusters lie inside the drift volume of their side: A: 0 <= z - shift <= z_max, C: -z_max <= z - shift <= 0
  const double lo = side > 0 ? zmax_hits - z_max : zmax_hits;
  const double hi = side > 0 ? zmin_hits : zmin_hits + z_max;
  double sh = zd;
  if (sh > hi) sh = hi;
  if (sh < lo) sh = lo;
  o.z_dca = (float)zd; o.z_shift = (float)sh; o.t0_us = (float)((double)side * sh / vdrift); o.dca_xy = (float)dca;
  return o;
}

// ---- O12-O13: legs of low-pT loopers and cluster tags ----
struct LegParams {
  float leg_min_qpt, leg_min_sinphi, leg_inner_min_sinphi, leg_apex_margin;
  int32_t leg_max_sector_gap, leg_inner_max_sector_gap;
  float leg_max_turn, leg_inner_max_turn, leg_centre_frac, leg_centre_abs, leg_radius_frac, leg_dz_max, leg_dzds_tol;
  float tag_qpt_low, tag_qpt_leg, tag_sinphi;
  int32_t ring;
};

// atan(r) for |r| <= 1: the degree-17 odd polynomial of Abramowitz & Stegun 4.4.49 (|error| <= 2e-8), Horner with fma.
inline float atan_unit(float r) {
  const float r2 = r * r;
  float p = 0.0028662257f;
  p = fma32(p, r2, -0.0161657367f);
  p = fma32(p, r2, 0.0429096138f);
  p = fma32(p, r2, -0.0752896400f);
  p = fma32(p, r2, 0.1065626393f);
  p = fma32(p, r2, -0.1420889944f);
  p = fma32(p, r2, 0.1999355085f);
  p = fma32(p, r2, -0.3333314528f);
  p = fma32(p, r2, 1.0f);
  return r * p;
}

// Angle of the vector (x, y) with y > 0, in (0, pi): octant reduction onto atan_unit.
inline float angle_upper(float y, float x) {
  const float half_pi = 1.57079632679f, pi = 3.14159265359f;
  if (std::fabs(x) <= y) return half_pi - atan_unit(x / y);
  if (x > 0.0f) return atan_unit(y / x);
  return pi + atan_unit(y / x);
}

struct LegEnd {  // an end of a merged track: the outer end in the frame of its outermost sector segment (sig = +1: the helix
  int32_t sector;  // continues along the fit direction), or the inner end in the frame of its innermost segment (sig = -1: against it)
  int32_t sig;
  float x, y, z, s, t, q;
  float c, R, xc, yc;  // cos(phi), radius, circle centre
  bool cand;
};

inline LegEnd leg_end(int sig, int sector, float x, float y, float z, float s, float t, float q, bool valid, float kq,
                      float x_last, const LegParams& L) {
  LegEnd e;
  e.sig = sig; e.sector = sector; e.x = x; e.y = y; e.z = z; e.s = s; e.t = t; e.q = q;
  e.c = 0; e.R = 0; e.xc = 0; e.yc = 0; e.cand = false;
  const float smin = sig > 0 ? L.leg_min_sinphi : L.leg_inner_min_sinphi;
  if (!valid || !(std::fabs(q) >= L.leg_min_qpt) || !(std::fabs(s) >= smin) || !(std::fabs(s) < 1.0f)) return e;
  const float k = q * kq;
  e.c = std::sqrt(fma32(-s, s, 1.0f));
  e.R = 1.0f / std::fabs(k);
  e.xc = x - s / k;
  e.yc = y + e.c / k;
  e.cand = sig < 0 || (e.xc + e.R) <= (x_last + L.leg_apex_margin);  // outer end: the helix turns back inside the TPC
  return e;
}

// Score of the pair (A, B) -- A is the track with the lower id, both ends of the same kind -- or a negative value if the
// helix continued from A does not arrive at B.  Everything is evaluated in A's frame; B's frame lies j sector steps ahead
// in A's turning sense.  For inner ends (sig = -1) the helix is continued AGAINST the fit direction: the turning sense and
// the slope change sign, the products of the two direction vectors do not.
inline float leg_pair_score(const LegEnd& A, const LegEnd& B, float kq, float ca, float sa, const LegParams& L) {
  if (!A.cand || !B.cand) return -1.0f;
  if (!(A.q * B.q < 0.0f)) return -1.0f;  // the two legs of a turn are fitted in opposite senses
  if (L.ring <= 0) { if (A.sector != B.sector) return -1.0f; }
  else if (A.sector / L.ring != B.sector / L.ring) return -1.0f;  // same z side
  if (A.sig != B.sig) return -1.0f;
  const float sig = (float)A.sig;
  const int sgn = ((sig * A.q) * kq > 0.0f) ? 1 : -1;  // sense in which the direction turns along the continuation
  // B's frame relative to A's: jrot sector steps (B's axis = A's axis + jrot * sector angle).  Over a turning point the
  // partner lies at most leg_max_sector_gap steps AHEAD in the turning sense; through the inner region the helix passes
  // near the beam line, where the azimuth of the position jumps by half a turn, so any sector of the side within
  // leg_inner_max_sector_gap steps either way is allowed.
  int jrot = 0;
  if (L.ring > 0) {
    const int dsec = ((B.sector - A.sector) % L.ring + L.ring) % L.ring;
    if (A.sig > 0) {
      const int j = ((dsec * sgn) % L.ring + L.ring) % L.ring;
      if (j > L.leg_max_sector_gap) return -1.0f;
      jrot = sgn * j;
    } else {
      jrot = (2 * dsec <= L.ring) ? dsec : dsec - L.ring;
      if (std::abs(jrot) > L.leg_inner_max_sector_gap) return -1.0f;
    }
  }
  // B's end point, centre and fit direction in A's frame: |jrot| rotations by the sector angle
  const float ss = (jrot >= 0) ? sa : -sa;
  const int nrot = std::abs(jrot);
  float bx = B.x, by = B.y, bxc = B.xc, byc = B.yc, bdx = B.c, bdy = B.s;
  for (int i = 0; i < nrot; i++) {
    float u = fma32(-by, ss, bx * ca), v = fma32(bx, ss, by * ca);
    bx = u; by = v;
    u = fma32(-byc, ss, bxc * ca); v = fma32(bxc, ss, byc * ca);
    bxc = u; byc = v;
    u = fma32(-bdy, ss, bdx * ca); v = fma32(bdx, ss, bdy * ca);
    bdx = u; bdy = v;
  }
  (void)bx; (void)by;
  // turning angle from A's fit direction to the reversed fit direction of B, in A's turning sense
  const float dot = -fma32(A.s, bdy, A.c * bdx);
  const float cross = fma32(A.s, bdx, -(A.c * bdy));
  const float yy = (float)sgn * cross;
  // turning angle in (0, 2 pi) in the turning sense; over a turning point it stays below half a turn (leg_max_turn < pi),
  // through the inner region it may be most of a turn
  const float two_pi = 6.28318530718f, pi = 3.14159265359f;
  float theta;
  if (yy > 0.0f) theta = angle_upper(yy, dot);
  else if (yy < 0.0f) theta = two_pi - angle_upper(-yy, dot);
  else if (dot < 0.0f) theta = pi;
  else return -1.0f;
  if (!(theta <= (A.sig > 0 ? L.leg_max_turn : L.leg_inner_max_turn))) return -1.0f;
  const float Rm = 0.5f * (A.R + B.R);
  const float arc = theta * Rm;
  const float dxc = A.xc - bxc, dyc = A.yc - byc;
  const float dc2 = fma32(dyc, dyc, dxc * dxc);
  const float tolc = fma32(L.leg_centre_frac, Rm, L.leg_centre_abs);
  const float tolc2 = tolc * tolc;
  if (!(dc2 <= tolc2)) return -1.0f;
  const float dR = A.R - B.R, tolR = L.leg_radius_frac * Rm;
  if (!(std::fabs(dR) <= tolR)) return -1.0f;
  const float tm = sig * (0.5f * (A.t - B.t));  // mean slope along the continuation
  const float dz = fma32(-tm, arc, B.z - A.z);
  if (!(std::fabs(dz) <= L.leg_dz_max)) return -1.0f;
  const float dt = A.t + B.t;
  if (!(std::fabs(dt) <= L.leg_dzds_tol)) return -1.0f;
  const float e1 = dc2 / tolc2, e2 = dR / tolR, e3 = dz / L.leg_dz_max, e4 = dt / L.leg_dzds_tol;
  float score = e1;
  score = fma32(e2, e2, score);
  score = fma32(e3, e3, score);
  score = fma32(e4, e4, score);
  return score;
}

void find_legs(Result* R, const Ctx& c, const LegParams& L) {
  const Params& P = c.P;
  const int nm = (int)R->merged.size(), nt = (int)R->tracks.size();
  const float th = P.tan_half_angle;
  const float den = fma32(th, th, 1.0f);
  const float ca = fma32(-th, th, 1.0f) / den, sa = (2.0f * th) / den;
  const float x_last = c.row_x[c.n_rows - 1];
  // ends of every merged track: outer = outer state (O8) of the last sector segment of its chain; inner = its own record
  std::vector<LegEnd> outer(nm), inner(nm);
  for (int m = 0; m < nm; m++) {
    const TrackRec& Mr = R->merged[m];
    const int head = Mr.pad[4];
    int tail = head;
    while (R->link_next[tail] >= 0) tail = R->link_next[tail];
    const KF& o = R->outer[tail];
    outer[m] = leg_end(+1, R->tracks[tail].sector, o.x, o.p[0], o.p[1] + R->outer_zref[tail], o.p[2], o.p[3], o.p[4],
                       R->tracks[tail].ndf >= 0, c.kq, x_last, L);
    inner[m] = leg_end(-1, Mr.sector, Mr.x, Mr.y, Mr.z, Mr.sinphi, Mr.dzds, Mr.qpt, R->tracks[head].ndf >= 0, c.kq, x_last, L);
  }
  // O12: best partner of every end among the ends of its kind (min by (score, id)), mutual pairs are linked
  auto match = [&](const std::vector<LegEnd>& ends, std::vector<int32_t>& partner) {
    std::vector<int32_t> best(nm, -1);
    std::vector<float> bs(nm, 0.0f);
    for (int a = 0; a < nm; a++) {
      if (!ends[a].cand) continue;
      for (int b = a + 1; b < nm; b++) {
        if (!ends[b].cand) continue;
        const float sc = leg_pair_score(ends[a], ends[b], c.kq, ca, sa, L);
        if (!(sc >= 0.0f)) continue;
        if (best[a] < 0 || sc < bs[a]) { best[a] = b; bs[a] = sc; }   // equal score: the lower id stays (b increases)
        if (best[b] < 0 || sc < bs[b]) { best[b] = a; bs[b] = sc; }   // equal score: the lower id stays (a increases)
      }
    }
    partner.assign(nm, -1);
    for (int a = 0; a < nm; a++) {
      const int b = best[a];
      if (b >= 0 && best[b] == a) partner[a] = b;
    }
  };
  match(outer, R->leg_partner);
  match(inner, R->leg_partner_in);
  // Legs joined at turning points (outer) and through the inner region (inner) form a chain along which |z| of the inner
  // ends grows (the particle drifts away from the side it was born on; the shift of a time frame is common to all legs).
  // The first leg is the one none of whose linked neighbours lies at a smaller |z| (equal |z|: the lower id).
  R->leg_first.assign(nm, 1);
  for (int a = 0; a < nm; a++) {
    const float za = std::fabs(R->merged[a].z);
    for (int kind = 0; kind < 2; kind++) {
      const int b = kind == 0 ? R->leg_partner[a] : R->leg_partner_in[a];
      if (b < 0) continue;
      const float zb = std::fabs(R->merged[b].z);
      if (zb < za || (zb == za && b < a)) R->leg_first[a] = 0;
    }
  }
  // O13: cluster tags
  R->cluster_tags.assign((size_t)R->n, 0);
  for (int t = 0; t < nt; t++) {
    const TrackRec& T = R->tracks[t];
    const int m = R->track_merged[t];
    const TrackRec& Mr = R->merged[m];
    uint8_t base = 0;
    if (std::fabs(Mr.qpt) > L.tag_qpt_low) base |= 1;
    if (R->leg_first[m] == 0 && std::fabs(Mr.qpt) > L.tag_qpt_leg) base |= 2;
    const float k = T.qpt * c.kq;
    for (int32_t h : R->track_hits[t]) {
      uint8_t f = base;
      if (T.ndf < 0) f |= 4;
      else {
        const float sl = fma32(c.cl[h].x - T.x, k, T.sinphi);  // sin(phi) is linear in x along a helix
        if (!(std::fabs(sl) <= L.tag_sinphi)) f |= 4;
      }
      R->cluster_tags[h] = f;
    }
  }
}

// ---- O14: one fit through both legs of a turn ("the refit was tuned to enable arbitrary rotations for
// following the full helix") ----
// The filter runs in a frame that is turned in sector steps whenever |sin(phi)| grows beyond fit_rot_sinphi, so that the
// track always points roughly along the frame's x axis -- also over the turning point, where no sector frame can describe
// it.  A hit of sector S seen from frame F (beta = (S - F) sector angles): its position is rotated into the frame; the
// pad row is no longer parallel to the frame's y axis, and the row coordinate of the track's crossing differs from the
// track's y at the hit's x by the factor D = cos(beta) + sin(beta) tan(phi), so the hit is a measurement of y with the
// error sigma_y * |D| (the dependence of D on the state is neglected, the z measurement is unchanged).
struct FitParams {
  float fit_rot_sinphi;   // turn the frame while |sin(phi)| exceeds this
  float fit_step_sinphi;  // a step never takes |sin(phi)| beyond this: it stops there and the frame is turned
  float fit_min_d;        // hits with |D| below this are not used (pad row nearly parallel to the track)
  float fit_reject_cut, shared_err_scale;
  int32_t ring;
};

struct ChainHit { int32_t h, sector; };

// cos / sin of n sector angles by n rotations of (1, 0)
inline void sector_cs(int n, float ca, float sa, float& cb, float& sb) {
  cb = 1.0f; sb = 0.0f;
  const float ss = (n >= 0) ? sa : -sa;
  for (int i = 0; i < std::abs(n); i++) {
    const float u = fma32(-sb, ss, cb * ca), v = fma32(cb, ss, sb * ca);
    cb = u; sb = v;
  }
}

// One pair: hits in trajectory order (first leg inner -> outer, second leg outer -> inner).  Returns false if a frame
// change or a transport fails.
bool fit_chain(const Ctx& c, const Result* R, const std::vector<ChainHit>& hits, float q0, const FitParams& F, float ca, float sa,
               KF& k, int& frame, float& z_ref, int& n_used, int& n_turn) {
  const Cl* cl = c.cl;
  const Params& P = c.P;
  const int n = (int)hits.size();
  const int ring = F.ring;  // <= 0: the frame cannot be turned (a fit that needs it fails)
  // start at the last hit, direction towards the one before it, in the last hit's sector frame
  const Cl& hN = cl[hits[n - 1].h];
  const Cl& hM = cl[hits[n - 2].h];
  if (hits[n - 1].sector != hits[n - 2].sector) return false;
  frame = hits[n - 1].sector;
  z_ref = hN.z;
  {
    const float dx = hM.x - hN.x, dy = hM.y - hN.y, dz = hM.z - hN.z;
    const float ds = std::sqrt(fma32(dx, dx, dy * dy));
    k.x = hN.x;
    k.p[0] = hN.y; k.p[1] = 0.0f; k.p[2] = dy / ds; k.p[3] = dz / ds; k.p[4] = q0;
  }
  n_turn = 0;
  for (int pass = 0; pass < 3; pass++) {
    reset_cov(k, P);
    n_used = 0;
    for (int j = 0; j < n; j++) {
      const int idx = (pass == 1) ? j : n - 1 - j;
      const Cl& h = cl[hits[idx].h];
      // Frame policy: keep the track roughly along the frame's x axis.  Turn the frame (one sector step at a time) while
      // |sin(phi)| > fit_rot_sinphi; if the way to the hit would take |sin(phi)| beyond fit_step_sinphi (the gap over the
      // turning point, where no pad row was tracked), go only as far as |sin(phi)| = fit_step_sinphi, turn, and go on.
      float cb = 1.0f, sb = 0.0f, X = 0.0f, Y = 0.0f;
      bool reached = false;
      for (int iter = 0; iter < 4 * ring + 1 && !reached; iter++) {
        for (int step = 0; step < ring && std::fabs(k.p[2]) > F.fit_rot_sinphi; step++) {
          const int sgn = k.p[2] > 0.0f ? 1 : -1;
          if (!rotate_frame(k, ca, (float)sgn * sa, c.kq, 0.9999f)) return false;
          frame = (frame / ring) * ring + ((frame % ring) + sgn + ring) % ring;
          n_turn++;
        }
        int beta = 0;
        if (ring > 0) {
          beta = ((hits[idx].sector - frame) % ring + ring) % ring;
          if (2 * beta > ring) beta -= ring;
        } else if (hits[idx].sector != frame) return false;
        sector_cs(beta, ca, sa, cb, sb);
        X = fma32(-h.y, sb, h.x * cb); Y = fma32(h.x, sb, h.y * cb);  // the hit in the fit frame
        const float kk = k.p[4] * c.kq;
        const float s_at = fma32(X - k.x, kk, k.p[2]);
        if (std::fabs(s_at) <= F.fit_step_sinphi) { reached = true; break; }
        const float target = s_at > 0.0f ? F.fit_step_sinphi : -F.fit_step_sinphi;
        const float dxp = (target - k.p[2]) / kk;
        if (!((dxp > 0.0f) == (X - k.x > 0.0f)) || dxp == 0.0f) return false;
        if (!transport(k, k.x + dxp, c.kq, P.max_sinphi)) return false;
      }
      if (!reached) return false;
      if (!transport(k, X, c.kq, P.max_sinphi)) return false;
      const float cphi = std::sqrt(fma32(-k.p[2], k.p[2], 1.0f));
      const float D = fma32(sb, k.p[2] / cphi, cb);
      if (!(std::fabs(D) >= F.fit_min_d)) continue;
      const bool sh = R->shared[hits[idx].h] != 0;
      const float ey = (sh ? P.sigma_y * F.shared_err_scale : P.sigma_y) * D;
      const float ez = sh ? P.sigma_z * F.shared_err_scale : P.sigma_z;
      const float vy = ey * ey, vz = ez * ez;
      const float iy = 1.0f / (k.C[0] + vy), iz = 1.0f / (k.C[2] + vz);
      const float dy = Y - k.p[0];
      const float dz = (h.z - z_ref) - k.p[1];
      const float d = fma32(dz * dz, iz, (dy * dy) * iy);
      if (!(d <= F.fit_reject_cut)) continue;
      update(k, Y, h.z - z_ref, vy, vz);
      n_used++;
    }
  }
  return true;
}

void fit_leg_pairs(Result* R, const Ctx& c, const FitParams& F) {
  const Params& P = c.P;
  const int nm = (int)R->merged.size();
  const float th = P.tan_half_angle;
  const float den = fma32(th, th, 1.0f);
  const float ca = fma32(-th, th, 1.0f) / den, sa = (2.0f * th) / den;
  R->leg_fits.clear();
  auto chain_hits = [&](int m, bool reversed, std::vector<ChainHit>& out) {
    std::vector<ChainHit> tmp;
    for (int t = R->merged[m].pad[4]; t >= 0; t = R->link_next[t])
      for (int32_t h : R->track_hits[t]) tmp.push_back({h, R->tracks[t].sector});
    if (reversed) std::reverse(tmp.begin(), tmp.end());
    out.insert(out.end(), tmp.begin(), tmp.end());
  };
  for (int a = 0; a < nm; a++) {
    const int b = R->leg_partner[a];
    if (b < a) continue;  // none, or the pair was done from its lower id
    const float za = std::fabs(R->merged[a].z), zb = std::fabs(R->merged[b].z);
    const bool a_first = (za < zb) || (za == zb);   // a < b: equal |z| -> the lower id
    const int f = a_first ? a : b, g = a_first ? b : a;
    std::vector<ChainHit> hits;
    chain_hits(f, false, hits);
    chain_hits(g, true, hits);
    TrackRec tr;
    std::memset(&tr, 0, sizeof(tr));
    KF k;
    k.x = 0; k.chi2 = 0;
    for (int i = 0; i < 5; i++) k.p[i] = 0;
    for (int i = 0; i < 15; i++) k.C[i] = 0;
    int frame = 0, n_used = 0, n_turn = 0;
    float z_ref = 0;
    bool ok = fit_chain(c, R, hits, R->merged[g].qpt, F, ca, sa, k, frame, z_ref, n_used, n_turn);
    // The filter arrives at the first leg's innermost hit running AGAINST that leg's direction of fit.  Report the state
    // as the leg's own record does -- direction outward, frame of the innermost segment's sector: seen from the frame
    // turned by half a ring the reversed direction has cos(phi) > 0 again (x, y, dz/ds and q/pT change sign, sin(phi) does
    // not), then the frame is turned step by step to the sector's.
    const int ring = F.ring;
    if (ok && ring > 0 && ring % 2 == 0) {
      static const float sg[5] = {-1.0f, 1.0f, 1.0f, -1.0f, -1.0f};
      k.x = -k.x; k.p[0] = -k.p[0]; k.p[3] = -k.p[3]; k.p[4] = -k.p[4];
      for (int i = 0; i < 5; i++)
        for (int j = 0; j <= i; j++) k.C[tri(i, j)] = (sg[i] * sg[j]) * k.C[tri(i, j)];
      frame = (frame / ring) * ring + ((frame % ring) + ring / 2) % ring;
      const int target = R->merged[f].sector;
      int dsec = ((target - frame) % ring + ring) % ring;
      if (2 * dsec > ring) dsec -= ring;
      const int sgn = dsec >= 0 ? 1 : -1;
      for (int i = 0; i < std::abs(dsec) && ok; i++) {
        ok = rotate_frame(k, ca, (float)sgn * sa, c.kq, 0.9999f);
        frame = (frame / ring) * ring + ((frame % ring) + sgn + ring) % ring;
      }
      // the fitted point left the pad row by (fitted - measured y) * sin(beta): a last, tiny step back onto it
      if (ok) ok = transport(k, c.cl[hits.front().h].x, c.kq, 0.9999f);
    }
    tr.sector = frame; tr.first_row = c.cl[hits.front().h].row; tr.last_row = c.cl[hits.back().h].row;
    tr.n_hits = (int32_t)hits.size();
    if (ok) {
      tr.x = k.x; tr.y = k.p[0]; tr.z = k.p[1] + z_ref; tr.sinphi = k.p[2]; tr.dzds = k.p[3]; tr.qpt = k.p[4];
      for (int i = 0; i < 15; i++) tr.cov[i] = k.C[i];
      tr.chi2 = k.chi2;
      tr.ndf = 2 * n_used - 5;
    } else {
      tr.ndf = -1;
    }
    tr.pad[0] = f; tr.pad[1] = g; tr.pad[2] = ok ? (int32_t)hits.size() - n_used : -1; tr.pad[3] = n_turn; tr.pad[4] = 0;
    R->leg_fits.push_back(tr);
  }
}

}  // namespace

extern "C" {

// Whole path O1-O7.  Returns an opaque result handle (free with orc_free).
void* orc_track(int32_t n_sectors, int32_t n_rows, const float* row_x, float bz, const Params* P, const Cl* cl,
                int64_t n, const int32_t* sector_offsets, int32_t brute) {
  Result* R = new Result;
  R->n = n; R->n_sectors = n_sectors; R->n_rows = n_rows;
  R->link_up_raw.assign(n, -1); R->link_down_raw.assign(n, -1);
  R->assignment.assign(n, -1);
  Ctx c = make_ctx(cl, row_x, n_rows, *P, bz, brute != 0);
  std::vector<Sector> secs(n_sectors);
  // O1: group by sector and row; canonical order inside a row slice
  for (int s = 0; s < n_sectors; s++) {
    Sector& S = secs[s];
    S.cl = cl;
    S.rows.assign(n_rows, {});
    for (int32_t i = sector_offsets[s]; i < sector_offsets[s + 1]; i++)
      if (cl[i].row >= 0 && cl[i].row < n_rows) S.rows[cl[i].row].push_back(i);
    for (auto& row : S.rows) std::sort(row.begin(), row.end(), [cl](int32_t a, int32_t b) { return key_less(cl, a, b); });
    find_neighbours(c, S, R->link_up_raw, R->link_down_raw);  // O2
  }
  // O3: keep mutual links only
  R->link_up = R->link_up_raw; R->link_down = R->link_down_raw;
  for (int64_t h = 0; h < n; h++) {
    const int32_t u = R->link_up_raw[h], d = R->link_down_raw[h];
    if (u >= 0 && R->link_down_raw[u] != h) R->link_up[h] = -1;
    if (d >= 0 && R->link_up_raw[d] != h) R->link_down[h] = -1;
  }
  // O4: start hits in (sector, key) order
  std::vector<int32_t> start_sector;
  for (int s = 0; s < n_sectors; s++)
    for (int r = 0; r < n_rows; r++)
      for (int32_t h : secs[s].rows[r])
        if (R->link_down[h] < 0 && R->link_up[h] >= 0) { R->start_hits.push_back(h); start_sector.push_back(s); }
  // O5: tracklets
  const size_t nt = R->start_hits.size();
  R->tracklets.resize(nt);
  R->row_hit.assign(nt * (size_t)n_rows, -1);
  std::vector<uint64_t> weight(n, 0);
  for (size_t t = 0; t < nt; t++) {
    Tracklet& T = R->tracklets[t];
    T.sector = start_sector[t]; T.start_hit = R->start_hits[t];
    int32_t* rh = &R->row_hit[t * (size_t)n_rows];
    build_tracklet(c, secs[T.sector], R->link_up, T.start_hit, T, rh);
    if (!T.valid) { for (int r = 0; r < n_rows; r++) rh[r] = -1; continue; }
    T.W = pack_weight(*P, T.n_hits, T.chi2, (uint32_t)t);
    for (int r = 0; r < n_rows; r++)
      if (rh[r] >= 0) weight[rh[r]] = std::max(weight[rh[r]], T.W);
  }
  // O6: selection by exclusive ownership; O7: refit
  std::vector<int32_t> hits;
  for (size_t t = 0; t < nt; t++) {
    const Tracklet& T = R->tracklets[t];
    if (!T.valid) continue;
    const int32_t* rh = &R->row_hit[t * (size_t)n_rows];
    hits.clear();
    for (int r = 0; r < n_rows; r++)
      if (rh[r] >= 0 && weight[rh[r]] == T.W) hits.push_back(rh[r]);
    if ((int)hits.size() < P->min_track_hits) continue;
    const int32_t id = (int32_t)R->tracks.size();
    for (int32_t h : hits) R->assignment[h] = id;
    TrackRec tr;
    std::memset(&tr, 0, sizeof(tr));
    tr.sector = T.sector; tr.first_row = cl[hits.front()].row; tr.last_row = cl[hits.back()].row;
    tr.n_hits = (int32_t)hits.size();
    KF k, ko; float z_ref = 0;
    ko.x = 0; ko.chi2 = 0;
    for (int i = 0; i < 5; i++) ko.p[i] = 0;
    for (int i = 0; i < 15; i++) ko.C[i] = 0;
    const bool ok = refit(c, hits, T.p[4], k, z_ref, &ko);
    R->track_hits.push_back(hits);
    R->outer.push_back(ko);
    R->outer_zref.push_back(z_ref);
    tr.x = k.x; tr.y = k.p[0]; tr.z = k.p[1] + z_ref; tr.sinphi = k.p[2]; tr.dzds = k.p[3]; tr.qpt = k.p[4];
    for (int i = 0; i < 15; i++) tr.cov[i] = k.C[i];
    tr.chi2 = k.chi2;
    tr.ndf = ok ? 2 * tr.n_hits - 5 : -1;
    R->tracks.push_back(tr);
    R->track_tracklet.push_back((int32_t)t);
  }
  // shared clusters (B7): a hit that the tracklet of an accepted track collected but lost to another owner
  R->shared.assign(n, 0);
  for (size_t k = 0; k < R->tracks.size(); k++) {
    const size_t t = (size_t)R->track_tracklet[k];
    const Tracklet& T = R->tracklets[t];
    const int32_t* rh = &R->row_hit[t * (size_t)n_rows];
    for (int r = 0; r < n_rows; r++)
      if (rh[r] >= 0 && weight[rh[r]] != T.W) R->shared[rh[r]] = 1;
  }
  return R;
}

// O8-O10 on a result of orc_track (same clusters, geometry and parameters).  Returns the number of merged tracks.
int64_t orc_merge(void* r, int32_t n_rows, const float* row_x, float bz, const Params* P, const Cl* cl, const MergeParams* M) {
  Result* R = (Result*)r;
  Ctx c = make_ctx(cl, row_x, n_rows, *P, bz, false);
  merge_tracks(R, c, *M);
  return (int64_t)R->merged.size();
}
const TrackRec* orc_merged(void* r) { return ((Result*)r)->merged.data(); }
const int32_t* orc_track_merged(void* r) { return ((Result*)r)->track_merged.data(); }
const int32_t* orc_link_next(void* r) { return ((Result*)r)->link_next.data(); }
const uint8_t* orc_shared(void* r) { return ((Result*)r)->shared.data(); }
// outer end of every sector track: x, y, z (absolute), sinphi, dzds, qpt, cov15 (21 floats per track)
void orc_outer(void* r, float* out21) {
  Result* R = (Result*)r;
  for (size_t t = 0; t < R->outer.size(); t++) {
    float* o = out21 + 21 * t;
    const KF& k = R->outer[t];
    o[0] = k.x; o[1] = k.p[0]; o[2] = k.p[1] + R->outer_zref[t]; o[3] = k.p[2]; o[4] = k.p[3]; o[5] = k.p[4];
    for (int i = 0; i < 15; i++) o[6 + i] = k.C[i];
  }
}

// O11 for every sector track (merged = 0) or merged track (merged = 1) of a result.  out: 4 floats per track.
void orc_time_estimate(void* r, int32_t merged, float bz, const Cl* cl, float vdrift, float z_max, float* out4) {
  Result* R = (Result*)r;
  const double kq = -((0.000299792458 * 10.0) * (double)bz);
  const int half = R->n_sectors / 2;
  const size_t n = merged ? R->merged.size() : R->tracks.size();
  for (size_t i = 0; i < n; i++) {
    const TrackRec& T = merged ? R->merged[i] : R->tracks[i];
    double zmin = 1e300, zmax = -1e300;
    for (int t = merged ? T.pad[4] : (int)i; t >= 0; t = merged ? R->link_next[t] : -1)
      for (int32_t h : R->track_hits[t]) { zmin = std::min(zmin, (double)cl[h].z); zmax = std::max(zmax, (double)cl[h].z); }
    const int side = (half > 0 && T.sector >= half) ? -1 : 1;
    const TimeRec o = time_estimate(T, kq, zmin, zmax, side, vdrift, z_max);
    out4[4 * i + 0] = o.z_dca; out4[4 * i + 1] = o.z_shift; out4[4 * i + 2] = o.t0_us; out4[4 * i + 3] = o.dca_xy;
  }
}
// O11 on a free-standing state (pins): state6 = x, y, z, sinphi, dzds, qpt
void orc_time_estimate_state(const float* state6, float bz, float zmin_hits, float zmax_hits, int32_t side, float vdrift,
                             float z_max, float* out4) {
  TrackRec T;
  std::memset(&T, 0, sizeof(T));
  T.x = state6[0]; T.y = state6[1]; T.z = state6[2]; T.sinphi = state6[3]; T.dzds = state6[4]; T.qpt = state6[5];
  const TimeRec o = time_estimate(T, -((0.000299792458 * 10.0) * (double)bz), zmin_hits, zmax_hits, side, vdrift, z_max);
  out4[0] = o.z_dca; out4[1] = o.z_shift; out4[2] = o.t0_us; out4[3] = o.dca_xy;
}


// O12-O13 on a result of orc_track + orc_merge.  Returns the number of leg links (pairs).
int64_t orc_legs(void* r, int32_t n_rows, const float* row_x, float bz, const Params* P, const Cl* cl, const LegParams* L) {
  Result* R = (Result*)r;
  Ctx c = make_ctx(cl, row_x, n_rows, *P, bz, false);
  find_legs(R, c, *L);
  int64_t n = 0;
  for (size_t m = 0; m < R->leg_partner.size(); m++)
    n += ((R->leg_partner[m] > (int32_t)m) ? 1 : 0) + ((R->leg_partner_in[m] > (int32_t)m) ? 1 : 0);
  return n;
}
const int32_t* orc_leg_partner(void* r) { return ((Result*)r)->leg_partner.data(); }
const int32_t* orc_leg_partner_in(void* r) { return ((Result*)r)->leg_partner_in.data(); }
const uint8_t* orc_leg_first(void* r) { return ((Result*)r)->leg_first.data(); }
const uint8_t* orc_cluster_tags(void* r) { return ((Result*)r)->cluster_tags.data(); }
float orc_angle_upper(float y, float x) { return angle_upper(y, x); }
// one end (sig = +1 outer, -1 inner): state7 = sector, x, y, z, sinphi, dzds, qpt -> out5 = cand, R, xc, yc, c
void orc_leg_end(int32_t sig, const float* state7, float bz, float x_last, const LegParams* L, float* out5) {
  const float kq = -((0.000299792458f * 10.0f) * bz);
  const LegEnd e = leg_end(sig, (int)state7[0], state7[1], state7[2], state7[3], state7[4], state7[5], state7[6], true, kq, x_last, *L);
  out5[0] = e.cand ? 1.0f : 0.0f; out5[1] = e.R; out5[2] = e.xc; out5[3] = e.yc; out5[4] = e.c;
}
// pair score of two ends of kind sig (A = first argument, taken as the lower id), or a negative value
float orc_leg_pair(int32_t sig, const float* a7, const float* b7, float bz, float x_last, float tan_half_angle, const LegParams* L) {
  const float kq = -((0.000299792458f * 10.0f) * bz);
  const float den = fma32(tan_half_angle, tan_half_angle, 1.0f);
  const float ca = fma32(-tan_half_angle, tan_half_angle, 1.0f) / den, sa = (2.0f * tan_half_angle) / den;
  const LegEnd A = leg_end(sig, (int)a7[0], a7[1], a7[2], a7[3], a7[4], a7[5], a7[6], true, kq, x_last, *L);
  const LegEnd B = leg_end(sig, (int)b7[0], b7[1], b7[2], b7[3], b7[4], b7[5], b7[6], true, kq, x_last, *L);
  return leg_pair_score(A, B, kq, ca, sa, *L);
}

// O14 on a result of orc_track + orc_merge + orc_legs.  Returns the number of pair fits (= outer links).
int64_t orc_fit_legs(void* r, int32_t n_rows, const float* row_x, float bz, const Params* P, const Cl* cl, const FitParams* F) {
  Result* R = (Result*)r;
  Ctx c = make_ctx(cl, row_x, n_rows, *P, bz, false);
  fit_leg_pairs(R, c, *F);
  return (int64_t)R->leg_fits.size();
}
const TrackRec* orc_leg_fits(void* r) { return ((Result*)r)->leg_fits.data(); }

void orc_free(void* r) { delete (Result*)r; }
int64_t orc_n_start(void* r) { return (int64_t)((Result*)r)->start_hits.size(); }
int64_t orc_n_tracks(void* r) { return (int64_t)((Result*)r)->tracks.size(); }
const int32_t* orc_link_up_raw(void* r) { return ((Result*)r)->link_up_raw.data(); }
const int32_t* orc_link_down_raw(void* r) { return ((Result*)r)->link_down_raw.data(); }
const int32_t* orc_link_up(void* r) { return ((Result*)r)->link_up.data(); }
const int32_t* orc_link_down(void* r) { return ((Result*)r)->link_down.data(); }
const int32_t* orc_start_hits(void* r) { return ((Result*)r)->start_hits.data(); }
const int32_t* orc_row_hit(void* r) { return ((Result*)r)->row_hit.data(); }
const int32_t* orc_assignment(void* r) { return ((Result*)r)->assignment.data(); }
const TrackRec* orc_tracks(void* r) { return ((Result*)r)->tracks.data(); }
const int32_t* orc_track_tracklet(void* r) { return ((Result*)r)->track_tracklet.data(); }
// tracklet table as flat arrays: ints (valid, first_row, last_row, n_hits) and floats (x, p5, C15, chi2, z_ref)
void orc_tracklets(void* r, int32_t* ints4, float* floats23) {
  Result* R = (Result*)r;
  for (size_t t = 0; t < R->tracklets.size(); t++) {
    const Tracklet& T = R->tracklets[t];
    ints4[4 * t + 0] = T.valid; ints4[4 * t + 1] = T.first_row; ints4[4 * t + 2] = T.last_row; ints4[4 * t + 3] = T.n_hits;
    float* f = floats23 + 23 * t;
    f[0] = T.x;
    for (int i = 0; i < 5; i++) f[1 + i] = T.p[i];
    for (int i = 0; i < 15; i++) f[6 + i] = T.C[i];
    f[21] = T.chi2; f[22] = T.z_ref;
  }
}

// ---- single-step entry points for the pins (P6-P8) ----
// state9: x, p[5]; cov15; returns 1 on success
int32_t orc_kf_transport(float* x, float* p5, float* cov15, float xnew, float bz, float max_sinphi) {
  KF k; k.x = *x; k.chi2 = 0;
  for (int i = 0; i < 5; i++) k.p[i] = p5[i];
  for (int i = 0; i < 15; i++) k.C[i] = cov15[i];
  const float kq = -((0.000299792458f * 10.0f) * bz);
  const bool ok = transport(k, xnew, kq, max_sinphi);
  *x = k.x;
  for (int i = 0; i < 5; i++) p5[i] = k.p[i];
  for (int i = 0; i < 15; i++) cov15[i] = k.C[i];
  return ok ? 1 : 0;
}
void orc_kf_update(float* p5, float* cov15, float* chi2, float ym, float zm, float sy2, float sz2) {
  KF k; k.x = 0; k.chi2 = *chi2;
  for (int i = 0; i < 5; i++) k.p[i] = p5[i];
  for (int i = 0; i < 15; i++) k.C[i] = cov15[i];
  update(k, ym, zm, sy2, sz2);
  for (int i = 0; i < 5; i++) p5[i] = k.p[i];
  for (int i = 0; i < 15; i++) cov15[i] = k.C[i];
  *chi2 = k.chi2;
}
// frame rotation by sgn * (sector angle) for the pins: state6 = x, y, z, sinphi, dzds, qpt
int32_t orc_rotate(float* x, float* p5, float* cov15, float tan_half_angle, int32_t sgn, float bz, float max_sinphi) {
  KF k; k.x = *x; k.chi2 = 0;
  for (int i = 0; i < 5; i++) k.p[i] = p5[i];
  for (int i = 0; i < 15; i++) k.C[i] = cov15[i];
  const float th = tan_half_angle;
  const float den = fma32(th, th, 1.0f);
  const float ca = fma32(-th, th, 1.0f) / den, sa = (2.0f * th) / den;
  const bool ok = rotate_frame(k, ca, (float)sgn * sa, -((0.000299792458f * 10.0f) * bz), max_sinphi);
  *x = k.x;
  for (int i = 0; i < 5; i++) p5[i] = k.p[i];
  for (int i = 0; i < 15; i++) cov15[i] = k.C[i];
  return ok ? 1 : 0;
}
// O7 on a free-standing hit list (hits in increasing x).  out: x, y, z, sinphi, dzds, qpt, cov15, chi2 (22 floats)
int32_t orc_refit_hits(int32_t n, const Cl* hits, float q0, float bz, const Params* P, float* out22) {
  std::vector<float> rx(1, 0.0f);
  Ctx c = make_ctx(hits, rx.data(), 1, *P, bz, true);
  std::vector<int32_t> idx(n);
  for (int i = 0; i < n; i++) idx[i] = i;
  KF k; float z_ref = 0;
  const bool ok = refit(c, idx, q0, k, z_ref);
  out22[0] = k.x; out22[1] = k.p[0]; out22[2] = k.p[1] + z_ref; out22[3] = k.p[2]; out22[4] = k.p[3]; out22[5] = k.p[4];
  for (int i = 0; i < 15; i++) out22[6 + i] = k.C[i];
  out22[21] = k.chi2;
  return ok ? 1 : 0;
}

}  // extern "C"
