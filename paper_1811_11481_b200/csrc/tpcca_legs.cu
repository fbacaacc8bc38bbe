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

// Outer end of a merged track, 48 bytes in the workspace: {z, s, t, q} {c, R, xc, yc} {sector, cand, -, -}
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
__global__ void __launch_bounds__(256) k_leg_reset(Dev d) {
  const int i = blockIdx.x * blockDim.x + threadIdx.x;
  if (i <= TPCCA_MAX_SECTORS) d.leg_sec[i] = 0;
  if (i < 4) d.leg_summary[i] = 0;
  if (i < d.cnt->n_merged) d.leg_best[i] = LEG_NONE;
}

__global__ void __launch_bounds__(128) k_leg_ends(Dev d) {
  const int m = blockIdx.x * blockDim.x + threadIdx.x;
  if (m >= d.cnt->n_merged) return;
  int tail = d.merged_out[m].pad[4];
  for (int nx = d.m_next[tail]; nx >= 0; nx = d.m_next[tail]) tail = nx;
  const tpcca_track_rec* tr = d.out_tracks;
  const float4* oa = reinterpret_cast<const float4*>(d.track_outer + (size_t)tail * 24);
  const float4 o0 = oa[0];  // x, y, z, sinphi
  const float4 o1 = oa[1];  // dzds, qpt, ..
  const float x = o0.x, y = o0.y, s = o0.w, t = o1.x, q = o1.y;
  const int sector = tr[tail].sector;
  float c = 0.f, R = 0.f, xc = 0.f, yc = 0.f;
  int cand = 0;
  if (tr[tail].ndf >= 0 && (fabsf(q) >= d.LP.leg_min_qpt) && (fabsf(s) >= d.LP.leg_min_sinphi) && (fabsf(s) < 1.0f)) {
    const float k = q * d.kq;
    c = sqrtf(fmaf(-s, s, 1.0f));
    R = 1.0f / fabsf(k);
    xc = x - s / k;
    yc = y + c / k;
    cand = ((xc + R) <= (d.row_x[d.n_rows - 1] + d.LP.leg_apex_margin)) ? 1 : 0;
  }
  float4* e = d.leg_ends + 3 * (size_t)m;
  e[0] = make_float4(o0.z, s, t, q);
  e[1] = make_float4(c, R, xc, yc);
  e[2] = make_float4(__int_as_float(sector), __int_as_float(cand), 0.f, 0.f);
  if (cand) atomicAdd(&d.leg_sec[sector + 1], 1);
}

// one block: exclusive scan of the (<= 64) per-sector counts; leg_sec[s] = start of sector s, cursors behind them
__global__ void __launch_bounds__(128) k_leg_offsets(Dev d) {
  __shared__ int sm[32];
  const int s = threadIdx.x;
  const int v = (s < TPCCA_MAX_SECTORS) ? d.leg_sec[s + 1] : 0;
  int tot;
  const int e = block_scan_excl(v, &tot, sm);
  __syncthreads();
  if (s < TPCCA_MAX_SECTORS) { d.leg_sec[s] = e; d.leg_cur[s] = e; }
  if (s == 0) d.leg_sec[TPCCA_MAX_SECTORS] = tot;
}

__global__ void __launch_bounds__(128) k_leg_scatter(Dev d) {
  const int m = blockIdx.x * blockDim.x + threadIdx.x;
  if (m >= d.cnt->n_merged) return;
  const float4 c = d.leg_ends[3 * (size_t)m + 2];
  if (!__float_as_int(c.y)) return;
  const int pos = atomicAdd(&d.leg_cur[__float_as_int(c.x)], 1);
  d.leg_list[pos] = m;  // order inside a sector is arbitrary: the match takes min (score, id)
}

// ---------------------------------------------------------------- (l1) pair scores (D4-D8): one warp per end A
// Every unordered pair is evaluated once, by the warp of the LOWER id, in A's frame; both ends receive the score through
// atomicMin of (score bits << 32 | partner id): min score, then lower partner id.
__device__ __forceinline__ float leg_pair_score(const Dev& d, const LegEnd& A, const LegEnd& B, int j, int sgn, float ca,
                                                float sa) {
  if (!(A.q * B.q < 0.0f)) return -1.0f;
  const float ss = (float)sgn * sa;
  float bxc = B.xc, byc = B.yc, bdx = B.c, bdy = B.s;
  for (int i = 0; i < j; i++) {
    float u = fmaf(-byc, ss, bxc * ca), v = fmaf(bxc, ss, byc * ca);
    bxc = u; byc = v;
    u = fmaf(-bdy, ss, bdx * ca); v = fmaf(bdx, ss, bdy * ca);
    bdx = u; bdy = v;
  }
  const float dot = -fmaf(A.s, bdy, A.c * bdx);
  const float cross = fmaf(A.s, bdx, -(A.c * bdy));
  const float yy = (float)sgn * cross;
  if (!(yy > 0.0f)) return -1.0f;
  const float theta = angle_upper(yy, dot);
  if (!(theta <= d.LP.leg_max_turn)) return -1.0f;
  const float Rm = 0.5f * (A.R + B.R);
  const float arc = theta * Rm;
  const float dxc = A.xc - bxc, dyc = A.yc - byc;
  const float dc2 = fmaf(dyc, dyc, dxc * dxc);
  const float tolc = fmaf(d.LP.leg_centre_frac, Rm, d.LP.leg_centre_abs);
  const float tolc2 = tolc * tolc;
  if (!(dc2 <= tolc2)) return -1.0f;
  const float dR = A.R - B.R, tolR = d.LP.leg_radius_frac * Rm;
  if (!(fabsf(dR) <= tolR)) return -1.0f;
  const float tm = 0.5f * (A.t - B.t);
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
  if (a >= d.cnt->n_merged) return;
  const LegEnd A = load_end(d.leg_ends, a);
  if (!A.cand) return;
  const float th = d.tan_half_angle;
  const float den = fmaf(th, th, 1.0f);
  const float ca = fmaf(-th, th, 1.0f) / den, sa = (2.0f * th) / den;
  const int ring = d.LP.ring;
  const int sgn = (A.q * d.kq > 0.0f) ? 1 : -1;
  const int base = ring > 0 ? (A.sector / ring) * ring : A.sector, l = A.sector - base;
  const int jmax = ring > 0 ? min(d.LP.leg_max_sector_gap, ring - 1) : 0;
  unsigned long long best = LEG_NONE;
  for (int j = 0; j <= jmax; j++) {
    const int sb = ring > 0 ? base + (((l + sgn * j) % ring) + ring) % ring : A.sector;
    if (sb >= d.n_sectors) continue;
    const int b0 = d.leg_sec[sb], b1 = d.leg_sec[sb + 1];
    for (int pos = b0 + lane; pos < b1; pos += 32) {
      const int b = d.leg_list[pos];
      if (b <= a) continue;
      const LegEnd B = load_end(d.leg_ends, b);
      const float sc = leg_pair_score(d, A, B, j, sgn, ca, sa);
      if (!(sc >= 0.0f)) continue;
      const unsigned long long sb64 = (unsigned long long)__float_as_uint(sc) << 32;  // score >= +0: bits order like values
      best = min(best, sb64 | (unsigned)b);
      atomicMin(&d.leg_best[b], sb64 | (unsigned)a);
    }
  }
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) {
    const unsigned long long v = __shfl_xor_sync(0xffffffffu, best, o);
    best = min(best, v);
  }
  if (lane == 0 && best != LEG_NONE) atomicMin(&d.leg_best[a], best);
}

// ---------------------------------------------------------------- (l2) mutual links, first leg (D9, D10)
__global__ void __launch_bounds__(256) k_leg_link(Dev d) {
  const int a = blockIdx.x * blockDim.x + threadIdx.x;
  if (a >= d.cnt->n_merged) return;
  int partner = -1;
  const unsigned long long ba = d.leg_best[a];
  if (ba != LEG_NONE) {
    const int b = (int)(ba & 0xffffffffull);
    const unsigned long long bb = d.leg_best[b];
    if (bb != LEG_NONE && (int)(bb & 0xffffffffull) == a) partner = b;
  }
  int first = 1;
  if (partner >= 0) {
    const float za = fabsf(d.merged_out[a].z), zb = fabsf(d.merged_out[partner].z);
    first = ((za < zb) || (za == zb && a < partner)) ? 1 : 0;
    if (a < partner) atomicAdd(&d.leg_summary[0], 1);
  }
  d.leg_partner_out[a] = partner;
  d.leg_first_out[a] = (uint8_t)first;
}

// ---------------------------------------------------------------- (l3) cluster tags (D11): one warp per sector track
__global__ void __launch_bounds__(128) k_leg_tags(Dev d) {
  const int lane = threadIdx.x & 31;
  const int t = (blockIdx.x * 128 + threadIdx.x) >> 5;
  if (t >= d.cnt->n_tracks) return;
  const tpcca_track_rec* T = &d.out_tracks[t];
  const int m = d.track_merged_out[t];
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
    if (n1) atomicAdd(&d.leg_summary[1], n1);
    if (n2) atomicAdd(&d.leg_summary[2], n2);
    if (n4) atomicAdd(&d.leg_summary[3], n4);
  }
}

__global__ void k_leg_summary(Dev d) {
  if (threadIdx.x < 4) d.leg_summary_out[threadIdx.x] = d.leg_summary[threadIdx.x];
}

void launch_legs(const Dev& d, Launch& L) {
  const int K = d.max_tracks;
  if (d.n > 0) cudaMemsetAsync(d.tags_out, 0, (size_t)d.n, L.st);
  if (d.n > 0 && K > 0) {
    k_leg_reset<<<(max(K, 128) + 255) / 256, 256, 0, L.st>>>(d);
    k_leg_ends<<<(K + 127) / 128, 128, 0, L.st>>>(d);
    k_leg_offsets<<<1, 128, 0, L.st>>>(d);
    k_leg_scatter<<<(K + 127) / 128, 128, 0, L.st>>>(d);
    k_leg_match<<<(K + 3) / 4, 128, 0, L.st>>>(d);
    k_leg_link<<<(K + 255) / 256, 256, 0, L.st>>>(d);
    k_leg_tags<<<(K + 3) / 4, 128, 0, L.st>>>(d);
    L.count += 7;
  } else {
    k_leg_reset<<<1, 256, 0, L.st>>>(d);
    L.count++;
  }
  k_leg_summary<<<1, 32, 0, L.st>>>(d);
  L.count++;
}
