// tpcca_legs.cu -- legs of low-pT loopers and cluster tags (steps O12-O13).
// PAPER.md:123 "additional legs of looping tracks do not point to the vertex ... special low-pT track merging";
// PAPER.md:157 clusters to remove for the compression: "very low-pT looping tracks below 50 MeV/c, additional legs of
// tracks below 200 MeV/c, and track segments with high inclination angle".
// Works on what the last tpcca_track + tpcca_merge left behind: the merged records, the chains (m_next), the outer ends
// written by k_refit (track_outer) and the owned-hit lists.  Arithmetic: DESIGN.md Table D, operation by operation.
#include "tpcca_dev.cuh"

#define LEG_NONE 0xffffffffffffffffull

// atan(r), |r| <= 1: Abramowitz & Stegun 4.4.49, Horner with one fma per coefficient (D6)
__device__ __forceinline__ float atan_unit(float r) {
  const float r2 = r * r;
  float p = 0.0028662257f;
  p = fmaf(p, r2, -0.0161657367f);
  p = fmaf(p, r2, 0.0429096138f);
  p = fmaf(p, r2, -0.0752896400f);
  p = fmaf(p, r2, 0.1065626393f);
  p = fmaf(p, r2, -0.1420889944f);
  p = fmaf(p, r2, 0.1999355085f);
  p = fmaf(p, r2, -0.3333314528f);
  p = fmaf(p, r2, 1.0f);
  return r * p;
}
// angle of (x, y), y > 0, in (0, pi)
__device__ __forceinline__ float angle_upper(float y, float x) {
  const float half_pi = 1.57079632679f, pi = 3.14159265359f;
  if (fabsf(x) <= y) return half_pi - atan_unit(x / y);
  if (x > 0.0f) return atan_unit(y / x);
  return pi + atan_unit(y / x);
}

// An end of a merged track, 48 bytes in the workspace: {z, s, t, q} {c, R, xc, yc} {sector, cand, -, -}.  Two kinds
// (D1): kind 0 = outer end (continued along the fit direction, sig = +1), kind 1 = inner end (against it, -1);
// kind-major arrays: entry kind * max_tracks + m.
struct LegEnd {
  float z, s, t, q, c, R, xc, yc;
  int sector, cand;
};
__device__ __forceinline__ LegEnd load_end(const float4* e, int m) {
  const float4 a = e[3 * m], b = e[3 * m + 1], c = e[3 * m + 2];
  LegEnd o;
  o.z = a.x; o.s = a.y; o.t = a.z; o.q = a.w; o.c = b.x; o.R = b.y; o.xc = b.z; o.yc = b.w;
  o.sector = __float_as_int(c.x); o.cand = __float_as_int(c.y);
  return o;
}

// ---------------------------------------------------------------- (l0) ends (D1-D3), candidate count per sector
// Candidates are bucketed by (sector, z bin of |z|): LEG_NZB bins of LEG_ZBIN cm per sector (the last one open-ended), so
// that an end only meets the partners inside a conservative z window (a search structure: any superset of the pairs that
// pass the cuts gives the same links).
#define LEG_NZB 128
#define LEG_ZBIN 32.0f
#define LEG_NKEY (TPCCA_MAX_SECTORS * LEG_NZB)
#define LEG_SEC_STRIDE (LEG_NKEY + 2)
__device__ __forceinline__ int leg_zbin(float z) {
  const float f = fabsf(z) * (1.0f / LEG_ZBIN);
  return (f < (float)(LEG_NZB - 1)) ? (int)f : LEG_NZB - 1;  // NaN -> last bin
}
__global__ void __launch_bounds__(256) k_leg_reset(Dev d) {
  const int i = blockIdx.x * blockDim.x + threadIdx.x;
  for (int j = i; j < 2 * LEG_SEC_STRIDE; j += gridDim.x * blockDim.x) d.leg_sec[j] = 0;
  if (i < 8) d.leg_summary[i] = 0;
  if (i < d.cnt->n_merged) { d.leg_best[i] = LEG_NONE; d.leg_best[d.max_tracks + i] = LEG_NONE; }
}

__device__ __forceinline__ void store_end(const Dev& d, int kind, int m, int sector, float x, float y, float z, float s, float t,
                                          float q, bool valid) {
  float c = 0.f, R = 0.f, xc = 0.f, yc = 0.f;
  int cand = 0;
  const float smin = kind == 0 ? d.LP.leg_min_sinphi : d.LP.leg_inner_min_sinphi;
  if (valid && (fabsf(q) >= d.LP.leg_min_qpt) && (fabsf(s) >= smin) && (fabsf(s) < 1.0f)) {
    const float k = q * d.kq;
    c = sqrtf(fmaf(-s, s, 1.0f));
    R = 1.0f / fabsf(k);
    xc = x - s / k;
    yc = y + c / k;
    cand = (kind == 1 || (xc + R) <= (d.row_x[d.n_rows - 1] + d.LP.leg_apex_margin)) ? 1 : 0;  // outer: turns back inside the TPC
  }
  float4* e = d.leg_ends + 3 * ((size_t)kind * d.max_tracks + m);
  e[0] = make_float4(z, s, t, q);
  e[1] = make_float4(c, R, xc, yc);
  e[2] = make_float4(__int_as_float(sector), __int_as_float(cand), 0.f, 0.f);
  if (cand) atomicAdd(&d.leg_sec[kind * LEG_SEC_STRIDE + sector * LEG_NZB + leg_zbin(z) + 1], 1);
}

__global__ void __launch_bounds__(128) k_leg_ends(Dev d) {
  const int m = blockIdx.x * blockDim.x + threadIdx.x;
  if (m >= d.cnt->n_merged) return;
  const tpcca_track_rec* tr = d.out_tracks;
  const tpcca_track_rec* M = &d.merged_out[m];
  const int head = M->pad[4];
  int tail = head;
  for (int nx = d.m_next[tail]; nx >= 0; nx = d.m_next[tail]) tail = nx;
  const float4* oa = reinterpret_cast<const float4*>(d.track_outer + (size_t)tail * 24);
  const float4 o0 = oa[0];  // x, y, z, sinphi
  const float4 o1 = oa[1];  // dzds, qpt, ..
  store_end(d, 0, m, tr[tail].sector, o0.x, o0.y, o0.z, o0.w, o1.x, o1.y, tr[tail].ndf >= 0);
  store_end(d, 1, m, M->sector, M->x, M->y, M->z, M->sinphi, M->dzds, M->qpt, tr[head].ndf >= 0);
}

// one block per kind: exclusive scan of the per-(sector, z bin) counts; leg_sec[key] = start of bucket key, cursors behind
__global__ void __launch_bounds__(1024) k_leg_offsets(Dev d) {
  __shared__ int sm[32];
  int32_t* sec = d.leg_sec + blockIdx.x * LEG_SEC_STRIDE;
  int32_t* cur = d.leg_cur + blockIdx.x * LEG_NKEY;
  int carry = 0;
  for (int k0 = 0; k0 < LEG_NKEY; k0 += 1024) {
    const int k = k0 + threadIdx.x;
    const int v = sec[k + 1];  // count of bucket k (read by all threads before anyone overwrites: the scan synchronises)
    int tot;
    const int e = block_scan_excl(v, &tot, sm);
    __syncthreads();
    sec[k] = carry + e;
    cur[k] = carry + e;
    carry += tot;
    __syncthreads();
  }
  if (threadIdx.x == 0) sec[LEG_NKEY] = carry;
}

__global__ void __launch_bounds__(128) k_leg_scatter(Dev d) {
  const int m = blockIdx.x * blockDim.x + threadIdx.x;
  const int kind = blockIdx.y;
  if (m >= d.cnt->n_merged) return;
  const float4* e = d.leg_ends + 3 * ((size_t)kind * d.max_tracks + m);
  const float4 c = e[2];
  if (!__float_as_int(c.y)) return;
  const float4 e0 = e[0];
  const int pos = atomicAdd(&d.leg_cur[kind * LEG_NKEY + __float_as_int(c.x) * LEG_NZB + leg_zbin(e0.x)], 1);
  d.leg_list[(size_t)kind * d.max_tracks + pos] = m;  // order inside a bucket is arbitrary: the match takes min (score, id)
  // the first 32 bytes of the record again, in bucket order: the lanes of k_leg_match read consecutive entries
  d.leg_bk[(size_t)(2 * kind) * d.max_tracks + pos] = e0;
  d.leg_bk[(size_t)(2 * kind + 1) * d.max_tracks + pos] = e[1];
}

// ---------------------------------------------------------------- (l1) pair scores (D4-D8): one warp per end A
// Every unordered pair is evaluated once, by the warp of the LOWER id, in A's frame; both ends receive the score through
// atomicMin of (score bits << 32 | partner id): min score, then lower partner id.
__device__ __forceinline__ float leg_pair_score(const Dev& d, const LegEnd& A, const LegEnd& B, int jrot, int sgn, float sig,
                                                float ca, float sa) {
  if (!(A.q * B.q < 0.0f)) return -1.0f;
  const float ss = (jrot >= 0) ? sa : -sa;
  const int nrot = abs(jrot);
  float bxc = B.xc, byc = B.yc, bdx = B.c, bdy = B.s;
  for (int i = 0; i < nrot; i++) {
    float u = fmaf(-byc, ss, bxc * ca), v = fmaf(bxc, ss, byc * ca);
    bxc = u; byc = v;
    u = fmaf(-bdy, ss, bdx * ca); v = fmaf(bdx, ss, bdy * ca);
    bdx = u; bdy = v;
  }
  const float dot = -fmaf(A.s, bdy, A.c * bdx);
  const float cross = fmaf(A.s, bdx, -(A.c * bdy));
  const float yy = (float)sgn * cross;
  const float two_pi = 6.28318530718f, pi = 3.14159265359f;
  float theta;
  if (yy > 0.0f) theta = angle_upper(yy, dot);
  else if (yy < 0.0f) theta = two_pi - angle_upper(-yy, dot);
  else if (dot < 0.0f) theta = pi;
  else return -1.0f;
  if (!(theta <= (sig > 0.0f ? d.LP.leg_max_turn : d.LP.leg_inner_max_turn))) return -1.0f;
  const float Rm = 0.5f * (A.R + B.R);
  const float arc = theta * Rm;
  const float dxc = A.xc - bxc, dyc = A.yc - byc;
  const float dc2 = fmaf(dyc, dyc, dxc * dxc);
  const float tolc = fmaf(d.LP.leg_centre_frac, Rm, d.LP.leg_centre_abs);
  const float tolc2 = tolc * tolc;
  if (!(dc2 <= tolc2)) return -1.0f;
  const float dR = A.R - B.R, tolR = d.LP.leg_radius_frac * Rm;
  if (!(fabsf(dR) <= tolR)) return -1.0f;
  const float tm = sig * (0.5f * (A.t - B.t));
  const float dz = fmaf(-tm, arc, B.z - A.z);
  if (!(fabsf(dz) <= d.LP.leg_dz_max)) return -1.0f;
  const float dt = A.t + B.t;
  if (!(fabsf(dt) <= d.LP.leg_dzds_tol)) return -1.0f;
  const float e1 = dc2 / tolc2, e2 = dR / tolR, e3 = dz / d.LP.leg_dz_max, e4 = dt / d.LP.leg_dzds_tol;
  float score = e1;
  score = fmaf(e2, e2, score);
  score = fmaf(e3, e3, score);
  score = fmaf(e4, e4, score);
  return score;
}

__global__ void __launch_bounds__(128) k_leg_match(Dev d) {
  const int lane = threadIdx.x & 31;
  const int a = (blockIdx.x * 128 + threadIdx.x) >> 5;
  const int kind = blockIdx.y;
  if (a >= d.cnt->n_merged) return;
  const float4* ends = d.leg_ends + 3 * (size_t)kind * d.max_tracks;
  const int32_t* sec = d.leg_sec + kind * LEG_SEC_STRIDE;
  const int32_t* list = d.leg_list + (size_t)kind * d.max_tracks;
  const float4* bk0 = d.leg_bk + (size_t)(2 * kind) * d.max_tracks;
  const float4* bk1 = d.leg_bk + (size_t)(2 * kind + 1) * d.max_tracks;
  unsigned long long* bestv = d.leg_best + (size_t)kind * d.max_tracks;
  const LegEnd A = load_end(ends, a);
  if (!A.cand) return;
  const float th = d.tan_half_angle;
  const float den = fmaf(th, th, 1.0f);
  const float ca = fmaf(-th, th, 1.0f) / den, sa = (2.0f * th) / den;
  const int ring = d.LP.ring;
  const float sig = kind == 0 ? 1.0f : -1.0f;
  const int sgn = ((sig * A.q) * d.kq > 0.0f) ? 1 : -1;
  const int base = ring > 0 ? (A.sector / ring) * ring : A.sector, l = A.sector - base;
  // Conservative z window of the partners (same z side, so |z| orders like z up to the sign): a partner passes
  // |tA + tB| <= dt_tol, |RA - RB| <= f Rm and theta <= theta_max, hence |mean slope| <= |tA| + dt_tol / 2 and
  // arc <= theta_max RA / (1 - f / 2); zB - zA lies within that product plus leg_dz_max.  1 % and one bin of slack.
  const float f2 = 0.5f * d.LP.leg_radius_frac;
  const float thmax = kind == 0 ? d.LP.leg_max_turn : d.LP.leg_inner_max_turn;
  int zb_lo = 0, zb_hi = LEG_NZB - 1;
  if (f2 < 0.9f) {
    const float reach = 1.01f * ((fabsf(A.t) + 0.5f * d.LP.leg_dzds_tol) * (thmax * A.R / (1.0f - f2)) + d.LP.leg_dz_max) + 1.0f;
    const float az = fabsf(A.z);
    zb_lo = max(0, leg_zbin(fmaxf(az - reach, 0.0f)) - 1);
    zb_hi = min(LEG_NZB - 1, leg_zbin(az + reach) + 1);
    if (!(reach == reach)) { zb_lo = 0; zb_hi = LEG_NZB - 1; }
  }
  // sector offsets dsec = 0 .. ring-1 of the partner; jrot as in DESIGN.md D4
  const int nsec = ring > 0 ? ring : 1;
  unsigned long long best = LEG_NONE;
  for (int dsec = 0; dsec < nsec; dsec++) {
    int jrot = 0;
    if (ring > 0) {
      if (kind == 0) {
        const int j = ((dsec * sgn) % ring + ring) % ring;
        if (j > d.LP.leg_max_sector_gap) continue;
        jrot = sgn * j;
      } else {
        jrot = (2 * dsec <= ring) ? dsec : dsec - ring;
        if (abs(jrot) > d.LP.leg_inner_max_sector_gap) continue;
      }
    }
    const int sb = ring > 0 ? base + (l + dsec) % ring : A.sector;
    if (sb >= d.n_sectors) continue;
    const int b0 = sec[sb * LEG_NZB + zb_lo], b1 = sec[sb * LEG_NZB + zb_hi + 1];
    for (int pos = b0 + lane; pos < b1; pos += 32) {
      const int b = list[pos];
      if (b <= a) continue;
      // the cheap cuts first, on the first 16 bytes of B's record (q/pT sign and slope sum), then the radius: the order of
      // the cuts does not change which pairs pass all of them (D7)
      const float4 b0v = bk0[pos];
      if (!(A.q * b0v.w < 0.0f) || !(fabsf(A.t + b0v.z) <= d.LP.leg_dzds_tol)) continue;
      const float4 b1v = bk1[pos];
      if (!(fabsf(A.R - b1v.y) <= d.LP.leg_radius_frac * (0.5f * (A.R + b1v.y)))) continue;
      LegEnd B;
      B.z = b0v.x; B.s = b0v.y; B.t = b0v.z; B.q = b0v.w; B.c = b1v.x; B.R = b1v.y; B.xc = b1v.z; B.yc = b1v.w;
      B.sector = sb; B.cand = 1;
      const float sc = leg_pair_score(d, A, B, jrot, sgn, sig, ca, sa);
      if (!(sc >= 0.0f)) continue;
      const unsigned long long sb64 = (unsigned long long)__float_as_uint(sc) << 32;  // score >= +0: bits order like values
      best = min(best, sb64 | (unsigned)b);
      atomicMin(&bestv[b], sb64 | (unsigned)a);
    }
  }
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) {
    const unsigned long long v = __shfl_xor_sync(0xffffffffu, best, o);
    best = min(best, v);
  }
  if (lane == 0 && best != LEG_NONE) atomicMin(&bestv[a], best);
}

// ---------------------------------------------------------------- (l2) mutual links, first leg (D9, D10)
__device__ __forceinline__ int mutual_partner(const unsigned long long* bestv, int a) {
  const unsigned long long ba = bestv[a];
  if (ba == LEG_NONE) return -1;
  const int b = (int)(ba & 0xffffffffull);
  const unsigned long long bb = bestv[b];
  return (bb != LEG_NONE && (int)(bb & 0xffffffffull) == a) ? b : -1;
}

__global__ void __launch_bounds__(256) k_leg_link(Dev d) {
  const int a = blockIdx.x * blockDim.x + threadIdx.x;
  if (a >= d.cnt->n_merged) return;
  const int po = mutual_partner(d.leg_best, a);
  const int pi = mutual_partner(d.leg_best + d.max_tracks, a);
  // first leg: no linked neighbour at a smaller |z| of the inner end (equal: the lower id), D10
  const float za = fabsf(d.merged_out[a].z);
  int first = 1;
  if (po >= 0) {
    const float zb = fabsf(d.merged_out[po].z);
    if (zb < za || (zb == za && po < a)) first = 0;
    if (a < po) atomicAdd(&d.leg_summary[0], 1);
  }
  if (pi >= 0) {
    const float zb = fabsf(d.merged_out[pi].z);
    if (zb < za || (zb == za && pi < a)) first = 0;
    if (a < pi) atomicAdd(&d.leg_summary[1], 1);
  }
  d.leg_partner_out[a] = po;
  d.leg_partner_in_out[a] = pi;
  d.leg_first_out[a] = (uint8_t)first;
}

// ---------------------------------------------------------------- (l3) cluster tags (D11): one warp per sector track
__global__ void __launch_bounds__(128) k_leg_tags(Dev d) {
  const int lane = threadIdx.x & 31;
  const int t = (blockIdx.x * 128 + threadIdx.x) >> 5;
  if (t >= d.cnt->n_tracks) return;
  const tpcca_track_rec* T = &d.out_tracks[t];
  const int m = d.track_merged_out[t];
  if (m < 0) return;  // a segment outside every chain (k_merge_reset's initial value): no merged record to read
  const float qm = fabsf(d.merged_out[m].qpt);
  int base = 0;
  if (qm > d.LP.tag_qpt_low) base |= 1;
  if (d.leg_first_out[m] == 0 && qm > d.LP.tag_qpt_leg) base |= 2;
  const float x0 = T->x, s0 = T->sinphi, k = T->qpt * d.kq;
  const bool failed = T->ndf < 0;
  const int2 wl = d.w_list[d.track_w[t]];
  int n1 = 0, n2 = 0, n4 = 0;
  for (int i = lane; i < wl.y; i += 32) {
    const int j = wl.x + i;
    int f = base;
    if (failed) f |= 4;
    else {
      const float sl = fmaf(d.row_x[d.th_row[j]] - x0, k, s0);  // sin(phi) is linear in x along a helix
      if (!(fabsf(sl) <= d.LP.tag_sinphi)) f |= 4;
    }
    d.tags_out[d.orig_idx[d.th_hit[j]]] = (uint8_t)f;
    n1 += f & 1; n2 += (f >> 1) & 1; n4 += (f >> 2) & 1;
  }
  n1 = __reduce_add_sync(0xffffffffu, n1); n2 = __reduce_add_sync(0xffffffffu, n2); n4 = __reduce_add_sync(0xffffffffu, n4);
  if (lane == 0) {
    if (n1) atomicAdd(&d.leg_summary[2], n1);
    if (n2) atomicAdd(&d.leg_summary[3], n2);
    if (n4) atomicAdd(&d.leg_summary[4], n4);
  }
}

__global__ void k_leg_summary(Dev d) {
  if (threadIdx.x < 8) d.leg_summary_out[threadIdx.x] = d.leg_summary[threadIdx.x];
}

void launch_legs(const Dev& d, Launch& L) {
  const int K = d.max_tracks;
  if (d.n > 0) cudaMemsetAsync(d.tags_out, 0, (size_t)d.n, L.st);
  if (d.n > 0 && K > 0) {
    k_leg_reset<<<(max(K, 2 * LEG_SEC_STRIDE) + 255) / 256, 256, 0, L.st>>>(d);
    k_leg_ends<<<(K + 127) / 128, 128, 0, L.st>>>(d);
    k_leg_offsets<<<2, 1024, 0, L.st>>>(d);
    k_leg_scatter<<<dim3((K + 127) / 128, 2), 128, 0, L.st>>>(d);
    k_leg_match<<<dim3((K + 3) / 4, 2), 128, 0, L.st>>>(d);
    k_leg_link<<<(K + 255) / 256, 256, 0, L.st>>>(d);
    k_leg_tags<<<(K + 3) / 4, 128, 0, L.st>>>(d);
    L.count += 7;
  } else {
    k_leg_reset<<<8, 256, 0, L.st>>>(d);
    L.count++;
  }
  k_leg_summary<<<1, 32, 0, L.st>>>(d);
  L.count++;
}

// ---------------------------------------------------------------- fit through both legs of a turn (O14)
// One lane per pair.  The hits of a leg are the owned-hit lists of its sector segments (chain order, increasing row).
#define FIT_MAX_SEGS 24  // sector segments per leg (as MERGE_MAX_SEGS: a merged chain grows in row, >= 10 rows per segment of 152)
struct FitSeg { int off, cnt, sector; };

__device__ __forceinline__ int ring_add(int frame, int step, int ring) {
  return (frame / ring) * ring + ((frame % ring) + step + ring) % ring;
}

// cos / sin of n sector angles by |n| rotations of (1, 0)
__device__ __forceinline__ void sector_cs(int n, float ca, float sa, float& cb, float& sb) {
  cb = 1.0f; sb = 0.0f;
  const float ss = (n >= 0) ? sa : -sa;
  for (int i = 0; i < abs(n); i++) {
    const float u = fmaf(-sb, ss, cb * ca), v = fmaf(cb, ss, sb * ca);
    cb = u; sb = v;
  }
}

struct FitCtx {
  KF k;
  int frame, n_used, n_turn;
  float z_ref;
  bool ok;
};

// one hit of the trajectory (E3-E5 of DESIGN.md section 15)
__device__ __forceinline__ void fit_hit(const Dev& d, FitCtx& c, float xh, float yh, float zh, int hsec, bool shared, float ca, float sa) {
  if (!c.ok) return;
  KF& k = c.k;
  const int ring = d.FP.ring;
  float cb = 1.0f, sb = 0.0f, X = 0.0f, Y = 0.0f;
  bool reached = false;
  for (int iter = 0; iter < 4 * ring + 1 && !reached; iter++) {
    for (int step = 0; step < ring && fabsf(k.s) > d.FP.fit_rot_sinphi; step++) {
      const int sgn = k.s > 0.0f ? 1 : -1;
      if (!kf_rotate(k, ca, (float)sgn * sa, d.kq, 0.9999f)) { c.ok = false; return; }
      c.frame = ring_add(c.frame, sgn, ring);
      c.n_turn++;
    }
    int beta = 0;
    if (ring > 0) {
      beta = ((hsec - c.frame) % ring + ring) % ring;
      if (2 * beta > ring) beta -= ring;
    } else if (hsec != c.frame) { c.ok = false; return; }
    sector_cs(beta, ca, sa, cb, sb);
    X = fmaf(-yh, sb, xh * cb); Y = fmaf(xh, sb, yh * cb);
    const float kk = k.q * d.kq;
    const float s_at = fmaf(X - k.x, kk, k.s);
    if (fabsf(s_at) <= d.FP.fit_step_sinphi) { reached = true; break; }
    const float target = s_at > 0.0f ? d.FP.fit_step_sinphi : -d.FP.fit_step_sinphi;
    const float dxp = (target - k.s) / kk;
    if (!((dxp > 0.0f) == (X - k.x > 0.0f)) || dxp == 0.0f) { c.ok = false; return; }
    if (!kf_transport(k, k.x + dxp, d.kq, d.P.max_sinphi)) { c.ok = false; return; }
  }
  if (!reached) { c.ok = false; return; }
  if (!kf_transport(k, X, d.kq, d.P.max_sinphi)) { c.ok = false; return; }
  const float cphi = sqrtf(fmaf(-k.s, k.s, 1.0f));
  const float D = fmaf(sb, k.s / cphi, cb);
  if (!(fabsf(D) >= d.FP.fit_min_d)) return;
  const float ey = (shared ? d.P.sigma_y * d.FP.shared_err_scale : d.P.sigma_y) * D;
  const float ez = shared ? d.P.sigma_z * d.FP.shared_err_scale : d.P.sigma_z;
  const float vy = ey * ey, vz = ez * ez;
  const float iy = 1.0f / (k.c00 + vy), iz = 1.0f / (k.c11 + vz);
  const float dy = Y - k.y;
  const float dz = (zh - c.z_ref) - k.z;
  const float dist = fmaf(dz * dz, iz, (dy * dy) * iy);
  if (!(dist <= d.FP.fit_reject_cut)) return;
  kf_update(k, Y, zh - c.z_ref, vy, vz, iy);
  c.n_used++;
}

__device__ __forceinline__ int leg_segments(const Dev& d, int m, FitSeg* segs) {
  int n = 0;
  int t = d.merged_out[m].pad[4];
  for (; t >= 0 && n < FIT_MAX_SEGS; t = d.m_next[t]) {
    const int2 wl = d.w_list[d.track_w[t]];
    segs[n].off = wl.x; segs[n].cnt = wl.y; segs[n].sector = d.out_tracks[t].sector;
    n++;
  }
  if (t >= 0) atomicOr(&d.cnt->status, TPCCA_STAT_CHAIN_TRUNCATED);
  return n;
}

__global__ void __launch_bounds__(64) k_leg_fit_flag(Dev d) {
  const int a = blockIdx.x * blockDim.x + threadIdx.x;
  if (a < d.cnt->n_merged) d.m_scan[a] = (d.leg_partner_out[a] > a) ? 1 : 0;
}

// The pairs are compacted (leg_list[slot] = lower merged id, slot = rank of the pair in id order = its output record) and
// fitted longest first (m_order: slots by decreasing hit count), so that a warp holds 32 pairs of about the same length
// instead of the few merged tracks in 32 that have a partner.  leg_list / m_order are free here: the first is rebuilt by
// every tpcca_find_legs, the second by every tpcca_merge.
__global__ void __launch_bounds__(64) k_leg_fit_list(Dev d) {
  const int a = blockIdx.x * blockDim.x + threadIdx.x;
  const int nm = d.cnt->n_merged;
  if (a == 0) d.leg_summary[6] = d.m_scan[nm];  // number of pairs, read by the order kernels
  if (a >= nm) return;
  const int b = d.leg_partner_out[a];
  if (b <= a) return;
  const int slot = d.m_scan[a];
  d.leg_list[slot] = a;
  d.leg_list[(size_t)d.max_tracks + slot] = (d.merged_out[a].n_hits + d.merged_out[b].n_hits) >> 1;  // sort key, clamped by the sort
}

__global__ void __launch_bounds__(64) k_leg_fit(Dev d) {
  const int p = blockIdx.x * blockDim.x + threadIdx.x;
  if (p >= d.leg_summary[6]) return;
  const int slot = d.m_order[p];
  const int a = d.leg_list[slot];
  const int b = d.leg_partner_out[a];
  const float za = fabsf(d.merged_out[a].z), zb = fabsf(d.merged_out[b].z);
  const bool a_first = (za < zb) || (za == zb);
  const int f = a_first ? a : b, g = a_first ? b : a;
  FitSeg sf[FIT_MAX_SEGS], sg[FIT_MAX_SEGS];
  const int nf = leg_segments(d, f, sf), ng = leg_segments(d, g, sg);
  const Rot R = sector_rotation(d.tan_half_angle);
  int n_total = 0;
  for (int i = 0; i < nf; i++) n_total += sf[i].cnt;
  for (int i = 0; i < ng; i++) n_total += sg[i].cnt;
  FitCtx c;
  c.ok = true; c.n_used = 0; c.n_turn = 0;
  // start: the last hit of the trajectory = the innermost hit of g's innermost segment, direction towards the hit before it
  const int jN = sg[0].off, jM = sg[0].off + 1;
  const float2 pN = d.th_yz[jN], pM = d.th_yz[jM];
  const float xN = d.row_x[d.th_row[jN]], xM = d.row_x[d.th_row[jM]];
  c.frame = sg[0].sector;
  c.z_ref = pN.y;
  {
    const float dx = xM - xN, dy = pM.x - pN.x, dz = pM.y - pN.y;
    const float ds = sqrtf(fmaf(dx, dx, dy * dy));
    c.k.x = xN;
    c.k.y = pN.x; c.k.z = 0.0f; c.k.s = dy / ds; c.k.t = dz / ds; c.k.q = d.merged_out[g].qpt;
    c.k.chi2 = 0.0f;
  }
  for (int pass = 0; pass < 3; pass++) {
    kf_reset_cov(c.k, d.P.cov0);
    c.n_used = 0;
    if (pass == 1) {  // forward along the trajectory: f inner -> outer, then g outer -> inner
      for (int si = 0; si < nf; si++)
        for (int i = 0; i < sf[si].cnt; i++) {
          const int j = sf[si].off + i;
          const float2 p = d.th_yz[j];
          fit_hit(d, c, d.row_x[d.th_row[j]], p.x, p.y, sf[si].sector, d.th_shared[j] != 0, R.ca, R.sa);
        }
      for (int si = ng - 1; si >= 0; si--)
        for (int i = sg[si].cnt - 1; i >= 0; i--) {
          const int j = sg[si].off + i;
          const float2 p = d.th_yz[j];
          fit_hit(d, c, d.row_x[d.th_row[j]], p.x, p.y, sg[si].sector, d.th_shared[j] != 0, R.ca, R.sa);
        }
    } else {          // backward: g inner -> outer, then f outer -> inner
      for (int si = 0; si < ng; si++)
        for (int i = 0; i < sg[si].cnt; i++) {
          const int j = sg[si].off + i;
          const float2 p = d.th_yz[j];
          fit_hit(d, c, d.row_x[d.th_row[j]], p.x, p.y, sg[si].sector, d.th_shared[j] != 0, R.ca, R.sa);
        }
      for (int si = nf - 1; si >= 0; si--)
        for (int i = sf[si].cnt - 1; i >= 0; i--) {
          const int j = sf[si].off + i;
          const float2 p = d.th_yz[j];
          fit_hit(d, c, d.row_x[d.th_row[j]], p.x, p.y, sf[si].sector, d.th_shared[j] != 0, R.ca, R.sa);
        }
    }
  }
  // report in the first leg's innermost sector frame, direction outward (E7)
  KF& k = c.k;
  const int ring = d.FP.ring;
  if (c.ok && ring > 0 && (ring & 1) == 0) {
    k.x = -k.x; k.y = -k.y; k.t = -k.t; k.q = -k.q;
    // sign pattern (-, +, +, -, -): an element changes sign iff exactly one of its indices is in {0, 3, 4}
    k.c10 = -k.c10; k.c20 = -k.c20; k.c31 = -k.c31; k.c32 = -k.c32; k.c41 = -k.c41; k.c42 = -k.c42;
    c.frame = ring_add(c.frame, ring / 2, ring);
    const int target = d.merged_out[f].sector;
    int dsec = ((target - c.frame) % ring + ring) % ring;
    if (2 * dsec > ring) dsec -= ring;
    const int sgn = dsec >= 0 ? 1 : -1;
    for (int i = 0; i < abs(dsec) && c.ok; i++) {
      c.ok = kf_rotate(k, R.ca, (float)sgn * R.sa, d.kq, 0.9999f);
      c.frame = ring_add(c.frame, sgn, ring);
    }
    if (c.ok) c.ok = kf_transport(k, d.row_x[d.th_row[sf[0].off]], d.kq, 0.9999f);
  }
  tpcca_track_rec o;
  memset(&o, 0, sizeof(o));
  o.sector = c.frame; o.first_row = d.th_row[sf[0].off]; o.last_row = d.th_row[sg[0].off]; o.n_hits = n_total;
  if (c.ok) {
    o.x = k.x; o.y = k.y; o.z = k.z + c.z_ref; o.sinphi = k.s; o.dzds = k.t; o.qpt = k.q;
    o.cov[0] = k.c00; o.cov[1] = k.c10; o.cov[2] = k.c11; o.cov[3] = k.c20; o.cov[4] = k.c21; o.cov[5] = k.c22;
    o.cov[6] = k.c30; o.cov[7] = k.c31; o.cov[8] = k.c32; o.cov[9] = k.c33; o.cov[10] = k.c40; o.cov[11] = k.c41;
    o.cov[12] = k.c42; o.cov[13] = k.c43; o.cov[14] = k.c44;
    o.chi2 = k.chi2;
    o.ndf = 2 * c.n_used - 5;
  } else {
    o.ndf = -1;
    atomicAdd(&d.leg_summary[5], 1);
  }
  o.pad[0] = f; o.pad[1] = g; o.pad[2] = c.ok ? n_total - c.n_used : -1; o.pad[3] = c.n_turn; o.pad[4] = 0;
  float4* dst = reinterpret_cast<float4*>(&d.fit_out[slot]);
  const float4* src = reinterpret_cast<const float4*>(&o);
#pragma unroll
  for (int i = 0; i < 8; i++) dst[i] = src[i];
}

// header: pairs = total of the flag scan (0 without tracks), failed fits counted in leg_summary[5]
__global__ void __launch_bounds__(1024) k_leg_fit_begin(Dev d) {
  if (threadIdx.x == 0) { d.leg_summary[5] = 0; d.leg_summary[6] = 0; }
  d.ord[4 * 1024 + threadIdx.x] = 0;  // counting-sort scratch of the pair order (slot 4: the merged fit is through with it)
}
__global__ void k_leg_fit_header(Dev d, int have_scan) {
  tpcca_out_header hd;
  hd.n_tracks = have_scan ? d.m_scan[d.cnt->n_merged] : 0;
  hd.n_tracklets = d.leg_summary[5]; hd.n_start_hits = 0; hd.status = d.cnt->status;
  *d.fit_hdr = hd;
}

void launch_leg_fit(const Dev& d, Launch& L) {
  const int K = d.max_tracks;
  k_leg_fit_begin<<<1, 1024, 0, L.st>>>(d);
  L.count++;
  const bool work = d.n > 0 && K > 0;
  if (work) {
    k_leg_fit_flag<<<(K + 63) / 64, 64, 0, L.st>>>(d);
    L.count++;
    launch_scan_i32(d.m_scan, &d.cnt->n_merged, K, d.scan_tmp, L);
    k_leg_fit_list<<<(K + 63) / 64, 64, 0, L.st>>>(d);
    L.count++;
    launch_order_desc(d, 4, d.leg_list + (size_t)K, &d.leg_summary[6], K, d.m_order, L);
    k_leg_fit<<<(K / 2 + 63) / 64, 64, 0, L.st>>>(d);  // at most K / 2 pairs
    L.count++;
  }
  k_leg_fit_header<<<1, 1, 0, L.st>>>(d, work ? 1 : 0);
  L.count++;
}
