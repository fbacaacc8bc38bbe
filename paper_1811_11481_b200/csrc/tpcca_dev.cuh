// tpcca_dev.cuh -- device-side context, layouts and fp32 helpers of the CUDA path.
// Arithmetic follows DESIGN.md "Arithmetic" (steps O2-O7) operation by operation; every translation
// unit is compiled with -fmad=false so that no multiply-add is contracted.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

#include "../../include/tpcca.h"

#define TPCCA_MAX_SECTORS 64
#define TPCCA_MAX_ROWS 256

struct __align__(16) GridHdr {  // 32 B per (sector,row) slice (read as two 16-byte words)
  float ymin, zmin, inv_by, inv_bz;
  int32_t ny, nz, bin_base, pad;  // pad = clusters in the slice
};

struct __align__(16) NbrHdr {  // 32 B per slice: the per-row constants of the neighbours finder (O2)
  int32_t su, sd;  // slices of the up / down row, -1 if none
  float t, wyu, wzu, wyd, wzd;
  int32_t pad;
};

struct DevCounters {  // device-resident scalars
  int32_t n_start;     // start hits (clamped to max_tracklets)
  int32_t n_tracks;    // accepted tracks (clamped to max_tracks)
  int32_t n_valid;     // non-void tracklets
  int32_t status;
  int32_t n_bins;      // total grid bins of the frame
  int32_t n_start_raw; // start hits before clamping to capacity
  int32_t n_work;      // seeds that reach the constructor (chain >= min_seed_hits)
  int32_t work_next[4];  // queue heads of the four tracklet-constructor kernels
  int32_t n_merged, n_links, n_fit_failed, pad0;  // merger (tpcca_merge)
  unsigned long long row_steps, searches, track_hits;  // work counters (roofline units)
  unsigned long long phase_steps[4];   // row steps of k_tl_e1 / e2 / e3a / e3b
  unsigned long long tracklet_hits;    // hits of all valid tracklets (one weight atomic each)
};

struct SecOff { int32_t v[TPCCA_MAX_SECTORS + 1]; };

// Everything a kernel needs, passed by value.
struct Dev {
  // geometry / parameters
  int32_t n_sectors, n_rows, n_slices;
  int32_t n_sm;  // multiprocessors of the handle's device (persistent grids are sized in multiples of it)
  float tan_half_angle, kq, sy2, sz2, inv_sy2, inv_sz2;
  tpcca_params P;
  const float* row_x;
  // per call
  const float4* clusters;
  int32_t n;
  // capacities
  int32_t max_tracklets, max_tracks, max_bins;
  // (a) grid
  int32_t* slice_count;    // [n_slices+1]
  int32_t* row_start;      // [n_slices+1] exclusive scan of slice_count
  uint32_t* slice_bbox;    // [n_slices*4] ordered-uint ymin, ymax, zmin, zmax
  GridHdr* grid;           // [n_slices]
  NbrHdr* nbr;             // [n_slices]
  int32_t* slice_fill;     // [n_slices+1] fill cursors of the slice scatter
  int32_t* bin_base;       // [n_slices+1] first bin of a slice (upper-bound layout from the slice counts)
  float4* srec;            // [n] clusters in slice order: (y, z, input index, -)
  int32_t* cluster_rank;   // [n] scratch (start-hit bucket keys, see sb_key)
  int32_t* bin_start;      // [max_bins+1] per slice at bin_base: start of every bin, then the slice end
  int32_t* scan_tmp;       // partial sums
  float2* yz;              // [n] sorted (sector,row,bin)
  int32_t* orig_idx;       // [n] sorted -> input index
  uint16_t* slice_of;      // [n] slice id of a sorted cluster
  // (b)-(d)
  int32_t* link_up;        // [n] sorted index space
  int32_t* link_down;
  int32_t* link_up_clean;
  uint8_t* shared_flag;    // [n] sorted index space: collected by the tracklet of an accepted track that does not own it
  int32_t* slice_nstart;   // [n_slices+1]
  int32_t* slice_sbase;    // [n_slices+1]
  int32_t* start_tmp;      // [n] start hits in arrival order
  int32_t* sb_key;         // [n] z-bucket of start_tmp[i] (global bucket id), aliases cluster_rank
  int32_t* sb_count;       // [max_tracklets+1] bucket histogram -> scan -> cursors
  int32_t* sb_sorted;      // [max_tracklets] start hits grouped by bucket
  int32_t* sb_skey;        // [max_tracklets] bucket of sb_sorted[p]
  int32_t* start_hits;     // [max_tracklets] canonical order (sorted indices)
  // (e)
  int32_t* seed_w;         // [max_tracklets+1] tracklet id t -> work index w, -1 for void seeds
  int32_t* ord;            // [4][1024] counting-sort scratch per order (0 refit, 1 E2, 2 E3a, 3 E3b): histogram [0,512), cursors [512,1024); zeroed per call
  int32_t* e_key;          // [3][max_tracklets] w-space sort keys (expected row steps) of the E2 / E3a / E3b work orders
  int32_t* e_order;        // [3][max_tracklets] E2 / E3a / E3b work orders: w by decreasing key
  int32_t* work_t;         // [max_tracklets] w -> t
  int32_t* row_hit;        // [max_tracklets][n_rows] indexed by w (dense over surviving seeds)
  float* tl_state;         // [max_tracklets][40] w-space: x, 5 parameters, 15 cov, chi2, row, status, ... (layout: k_tl_e3a)
  int32_t* tl_ints;        // [max_tracklets][4] valid, first_row, last_row, n_hits
  float* tl_floats;        // [max_tracklets][8] x, y, z~, sinphi, dzds, qpt, chi2, z_ref
  unsigned long long* tl_W;        // [max_tracklets]
  unsigned long long* hit_weight;  // [n]
  // (f),(g)
  int32_t* sel_scan;       // [max_tracklets+1] t-space: accept flag -> exclusive scan = track id
  int32_t* tl_track;       // [max_tracklets] t-space: track id or -1 (only read for tracklets that own hits)
  int32_t* track_tracklet; // [max_tracks] track id -> t
  int32_t* track_w;        // [max_tracks] track id -> w
  int32_t* track_order;    // [max_tracks] refit order: track ids by decreasing hit count
  int32_t* track_len;      // [max_tracks] hit count of track id (sort key of the refit order)
  int2* w_list;            // [max_tracklets] w-space, accepted tracklets: (offset, count) of the owned-hit list
  float2* th_yz;           // [n] owned-hit lists (innermost first): (y, z)
  uint8_t* th_row;         // [n] their rows
  int32_t* th_hit;         // [n] their sorted cluster indices
  uint8_t* th_shared;      // [n] their shared flags (filled by tpcca_merge)
  float* track_outer;      // [max_tracks][24] outer end of every track: x, y, z, sinphi, dzds, qpt, cov15 (after refit pass 2)
  // merger
  tpcca_merge_params MP;
  unsigned long long* m_best_out;  // [max_tracks] (chi2 bits << 32 | partner id), ~0 = none
  unsigned long long* m_best_in;
  int32_t* m_next;         // [max_tracks] continuation of a sector track or -1
  int32_t* m_prev;
  int32_t* m_scan;         // [max_tracks+1] head flag -> exclusive scan = merged id
  int32_t* m_head;         // [max_tracks] merged id -> head sector track
  int32_t* m_len;          // [max_tracks] merged id -> total hits (fit work order key)
  int32_t* m_order;        // [max_tracks] merged ids by decreasing length
  int2* m_cand;            // [max_tracks] inner ends bucketed by (sector, first_row): (z bits, track id)
  tpcca_out_header* merged_hdr;
  tpcca_track_rec* merged_out;
  int32_t* track_merged_out;
  // looper legs and cluster tags (tpcca_find_legs)
  tpcca_leg_params LP;
  float4* leg_ends;                // [2][max_tracks][3] outer / inner end of every merged track (layout: tpcca_legs.cu)
  unsigned long long* leg_best;    // [2][max_tracks] (score bits << 32 | partner id), ~0 = none
  int32_t* leg_sec;                // [2][TPCCA_MAX_SECTORS*128+2] candidate ends per (sector, z bin) -> bucket starts
  int32_t* leg_cur;                // [2][TPCCA_MAX_SECTORS*128] scatter cursors
  int32_t* leg_list;               // [2][max_tracks] candidate ends grouped by (sector, z bin)
  float4* leg_bk;                  // [2][2][max_tracks] first 32 bytes of the candidates' records, in leg_list order
  int32_t* leg_summary;            // [8] links per kind, tagged clusters per bit
  int32_t* leg_partner_out;
  int32_t* leg_partner_in_out;
  uint8_t* leg_first_out;
  uint8_t* tags_out;
  int32_t* leg_summary_out;
  // fit through both legs of a turn (tpcca_fit_legs)
  tpcca_leg_fit_params FP;
  tpcca_out_header* fit_hdr;
  tpcca_track_rec* fit_out;
  DevCounters* cnt;
  tpcca_out_header* out_hdr;
  tpcca_track_rec* out_tracks;
  int32_t* out_assign;
};

__device__ __forceinline__ uint32_t ordf(float f) {
  const uint32_t b = __float_as_uint(f);
  return (b & 0x80000000u) ? ~b : (b | 0x80000000u);
}
__device__ __forceinline__ float unordf(uint32_t o) {
  return __uint_as_float((o & 0x80000000u) ? (o & 0x7FFFFFFFu) : ~o);
}

__device__ __forceinline__ int sector_of(const SecOff& so, int n_sectors, int i) {
  int lo = 0, hi = n_sectors;  // so.v[lo] <= i < so.v[hi]
  while (hi - lo > 1) {
    const int mid = (lo + hi) >> 1;
    if (so.v[mid] <= i) lo = mid; else hi = mid;
  }
  return lo;
}

// ---- Kalman state ----
struct KF {
  float x;
  float y, z, s, t, q;  // y, z~ = z - z_ref, sin(phi), dz/ds, q/pT
  float c00, c10, c11, c20, c21, c22, c30, c31, c32, c33, c40, c41, c42, c43, c44;
  float chi2;
};

__device__ __forceinline__ void kf_reset_cov(KF& k, const float* cov0) {
  k.c00 = cov0[0]; k.c11 = cov0[1]; k.c22 = cov0[2]; k.c33 = cov0[3]; k.c44 = cov0[4];
  k.c10 = k.c20 = k.c21 = k.c30 = k.c31 = k.c32 = k.c40 = k.c41 = k.c42 = k.c43 = 0.0f;
  k.chi2 = 0.0f;
}

// Transport x -> xnew.  false: |sin(phi)| would exceed max_sinphi (state unchanged).
// DESIGN.md section 3 "Transport": every fmaf below is a fused operation the section states (nothing else fuses:
// the translation units are compiled with -fmad=false).  C <- F C F^T is the 51-fma expansion of M = F C, C' = M F^T.
__device__ __forceinline__ bool kf_transport(KF& k, float xnew, float kq, float max_sinphi) {
  const float dx = xnew - k.x;
  if (dx == 0.0f) return true;
  const float s = k.s, t = k.t;
  const float kk = k.q * kq;
  const float s1 = fmaf(dx, kk, s);
  if (!(fabsf(s) <= max_sinphi) || !(fabsf(s1) <= max_sinphi)) return false;
  const float c0 = sqrtf(fmaf(-s, s, 1.0f));
  const float c1 = sqrtf(fmaf(-s1, s1, 1.0f));
  const float cc = c0 + c1;
  const float c01 = c0 * c1;
  const float inv = 1.0f / (c01 * cc);  // the one division shared by 1/cc, 1/c0, 1/c1
  const float icc = c01 * inv, ic0 = (c1 * cc) * inv, ic1 = (c0 * cc) * inv;
  const float f = (s + s1) * icc;
  const float dy = dx * f;
  float L = sqrtf(fmaf(dx, dx, dy * dy));
  if (dx < 0.0f) L = -L;
  const float u = (0.5f * kk) * L;
  const float u2 = u * u;
  const float g = fmaf(u2, fmaf(u2, 0.075f, 0.16666667f), 1.0f);
  const float dS = L * g;
  const float fs0 = fmaf(f * s, ic0, 1.0f) * icc;
  const float fs1 = fmaf(f * s1, ic1, 1.0f) * icc;
  const float h = dx * kq;
  const float fss = fs0 + fs1;
  const float a02 = dx * fss;
  const float a04 = (dx * fs1) * h;
  const float w = (t * g) * ((dx * dy) / L);
  const float a12 = w * fss;
  const float a13 = dS;
  const float a14 = (w * fs1) * h;
  const float a24 = h;
  k.y = k.y + dy;
  k.z = fmaf(t, dS, k.z);
  k.s = s1;
  k.x = xnew;
  const float c00 = k.c00, c10 = k.c10, c11 = k.c11, c20 = k.c20, c21 = k.c21, c22 = k.c22, c30 = k.c30,
              c31 = k.c31, c32 = k.c32, c33 = k.c33, c40 = k.c40, c41 = k.c41, c42 = k.c42, c43 = k.c43, c44 = k.c44;
  // M = F C  (rows 3 and 4 of F are unit rows: M_3j = C_3j, M_4j = C_4j)
  const float m00 = fmaf(a04, c40, fmaf(a02, c20, c00));
  const float m02 = fmaf(a04, c42, fmaf(a02, c22, c20));
  const float m04 = fmaf(a04, c44, fmaf(a02, c42, c40));
  const float m10 = fmaf(a14, c40, fmaf(a13, c30, fmaf(a12, c20, c10)));
  const float m11 = fmaf(a14, c41, fmaf(a13, c31, fmaf(a12, c21, c11)));
  const float m12 = fmaf(a14, c42, fmaf(a13, c32, fmaf(a12, c22, c21)));
  const float m13 = fmaf(a14, c43, fmaf(a13, c33, fmaf(a12, c32, c31)));
  const float m14 = fmaf(a14, c44, fmaf(a13, c43, fmaf(a12, c42, c41)));
  const float m20 = fmaf(a24, c40, c20);
  const float m21 = fmaf(a24, c41, c21);
  const float m22 = fmaf(a24, c42, c22);
  const float m23 = fmaf(a24, c43, c32);
  const float m24 = fmaf(a24, c44, c42);
  // C' = M F^T, lower triangle
  k.c00 = fmaf(a04, m04, fmaf(a02, m02, m00));
  k.c10 = fmaf(a04, m14, fmaf(a02, m12, m10));
  k.c11 = fmaf(a14, m14, fmaf(a13, m13, fmaf(a12, m12, m11)));
  k.c20 = fmaf(a04, m24, fmaf(a02, m22, m20));
  k.c21 = fmaf(a14, m24, fmaf(a13, m23, fmaf(a12, m22, m21)));
  k.c22 = fmaf(a24, m24, m22);
  k.c30 = fmaf(a04, c43, fmaf(a02, c32, c30));
  k.c31 = fmaf(a14, c43, fmaf(a13, c33, fmaf(a12, c32, c31)));
  k.c32 = fmaf(a24, c43, c32);
  k.c40 = fmaf(a04, c44, fmaf(a02, c42, c40));
  k.c41 = fmaf(a14, c44, fmaf(a13, c43, fmaf(a12, c42, c41)));
  k.c42 = fmaf(a24, c44, c42);
  return true;
}

// One scalar measurement update of component with pre-update column (i0..i4), state value xi, variance v
// (x_j <- fma(K_j, r, x_j), C_jl <- fma(-K_j, ci_l, C_jl), chi2 <- fma(r*r, w, chi2)).
__device__ __forceinline__ void kf_update1(KF& k, float i0, float i1, float i2, float i3, float i4, float r, float w) {
  const float K0 = i0 * w, K1 = i1 * w, K2 = i2 * w, K3 = i3 * w, K4 = i4 * w;
  k.y = fmaf(K0, r, k.y); k.z = fmaf(K1, r, k.z); k.s = fmaf(K2, r, k.s); k.t = fmaf(K3, r, k.t); k.q = fmaf(K4, r, k.q);
  k.c00 = fmaf(-K0, i0, k.c00);
  k.c10 = fmaf(-K1, i0, k.c10); k.c11 = fmaf(-K1, i1, k.c11);
  k.c20 = fmaf(-K2, i0, k.c20); k.c21 = fmaf(-K2, i1, k.c21); k.c22 = fmaf(-K2, i2, k.c22);
  k.c30 = fmaf(-K3, i0, k.c30); k.c31 = fmaf(-K3, i1, k.c31); k.c32 = fmaf(-K3, i2, k.c32); k.c33 = fmaf(-K3, i3, k.c33);
  k.c40 = fmaf(-K4, i0, k.c40); k.c41 = fmaf(-K4, i1, k.c41); k.c42 = fmaf(-K4, i2, k.c42); k.c43 = fmaf(-K4, i3, k.c43);
  k.c44 = fmaf(-K4, i4, k.c44);
  k.chi2 = fmaf(r * r, w, k.chi2);
}

// Sequential scalar updates, y then z~; w = 1/S of each.  wy: the caller's 1 / (c00 + sy2) if it already has it (the predicted
// distance of a hit uses the same quotient), else a negative value.
__device__ __forceinline__ void kf_update(KF& k, float ym, float zm, float sy2, float sz2, float wy = -1.0f) {
  if (wy < 0.0f) wy = 1.0f / (k.c00 + sy2);
  kf_update1(k, k.c00, k.c10, k.c20, k.c30, k.c40, ym - k.y, wy);                     // component 0: column (c00, c10, c20, c30, c40)
  kf_update1(k, k.c10, k.c11, k.c21, k.c31, k.c41, zm - k.z, 1.0f / (k.c11 + sz2));  // component 1: column (c10, c11, c21, c31, c41)
}

// ---- sector frames (used by the merger and by the fit through both legs of a turn) ----
struct Rot {  // cos and sin of the sector angle from tan(10 deg) by the double-angle formulas
  float ca, sa;
};
__device__ __forceinline__ Rot sector_rotation(float th) {
  const float den = fmaf(th, th, 1.0f);
  Rot r;
  r.ca = fmaf(-th, th, 1.0f) / den;
  r.sa = (2.0f * th) / den;
  return r;
}

// Frame change by sgn * (sector angle): ss = sgn * sin.  false: |sin(phi)| leaves the allowed range (state unchanged).
__device__ __forceinline__ bool kf_rotate(KF& k, float ca, float ss, float kq, float max_sinphi) {
  const float s = k.s;
  if (!(fabsf(s) <= max_sinphi)) return false;
  const float cphi = sqrtf(fmaf(-s, s, 1.0f));
  const float s1 = fmaf(s, ca, -(cphi * ss));
  if (!(fabsf(s1) <= max_sinphi)) return false;
  const float c1 = sqrtf(fmaf(-s1, s1, 1.0f));
  const float rr = c1 / cphi;
  const float ry = cphi / c1;
  const float rz = -((k.t * ss) / c1);
  const float rs = -((k.q * kq) * ss);
  const float x = k.x, y = k.y;
  k.x = fmaf(y, ss, x * ca);
  k.y = fmaf(y, ca, -(x * ss));
  k.s = s1;
  // M = F C with F = diag(ry, 1, rr, 1, 1) + rz at (1,0) + rs at (2,0); C' = M F^T
  const float m00 = ry * k.c00;
  const float m10 = fmaf(rz, k.c00, k.c10), m11 = fmaf(rz, k.c10, k.c11);
  const float m20 = fmaf(rs, k.c00, rr * k.c20), m21 = fmaf(rs, k.c10, rr * k.c21), m22 = fmaf(rs, k.c20, rr * k.c22);
  const float m30 = k.c30, m31 = k.c31, m32 = k.c32;
  const float m40 = k.c40, m41 = k.c41, m42 = k.c42;
  k.c00 = m00 * ry;
  k.c10 = m10 * ry; k.c11 = fmaf(rz, m10, m11);
  k.c20 = m20 * ry; k.c21 = fmaf(rz, m20, m21); k.c22 = fmaf(rs, m20, m22 * rr);
  k.c30 = m30 * ry; k.c31 = fmaf(rz, m30, m31); k.c32 = fmaf(rs, m30, m32 * rr);
  k.c40 = m40 * ry; k.c41 = fmaf(rz, m40, m41); k.c42 = fmaf(rs, m40, m42 * rr);
  return true;
}

__device__ __forceinline__ int ring_neighbour(int sector, int side, int ring) {
  if (ring <= 0) return -1;
  const int base = (sector / ring) * ring, l = sector - base;
  return base + (l + side + ring) % ring;
}

// same-row key order (ord z, ord y, input index): true if a < b
__device__ __forceinline__ bool key_less(float za, float ya, int32_t ia, float zb, float yb, int32_t ib) {
  const uint32_t oza = ordf(za), ozb = ordf(zb);
  if (oza != ozb) return oza < ozb;
  const uint32_t oya = ordf(ya), oyb = ordf(yb);
  if (oya != oyb) return oya < oyb;
  return ia < ib;
}

// Conservative bin range of [lo, hi] along one grid axis (monotone fp32 map + clamp => superset).
__device__ __forceinline__ void bin_range(float lo, float hi, float vmin, float inv_b, int nb, int& b0, int& b1) {
  const float f0 = (lo - vmin) * inv_b, f1 = (hi - vmin) * inv_b;
  b0 = (f0 > 0.0f) ? ((f0 < (float)nb) ? (int)f0 : nb - 1) : 0;
  b1 = (f1 >= 0.0f) ? ((f1 < (float)nb) ? (int)f1 : nb - 1) : -1;  // -1 => empty range
  if (!(lo <= hi)) { b0 = 1; b1 = 0; }                             // NaN window: nothing
}

// Conservative bin range with the clamps done in the float domain (any superset of the window is a valid search
// structure, O1): b0 = bin of lo clamped to [0, nb-1]; b1 = bin of hi clamped to nb-1, or -1 below the grid.
__device__ __forceinline__ void bin_range_fast(float lo, float hi, float vmin, float inv_b, int nb, int& b0, int& b1) {
  const float top = (float)(nb - 1);
  const float f0 = (lo - vmin) * inv_b, f1 = (hi - vmin) * inv_b;
  b0 = (int)fminf(fmaxf(f0, 0.0f), top);            // NaN -> 0
  b1 = (f1 >= 0.0f) ? (int)fminf(f1, top) : -1;      // NaN -> -1 (empty)
}

// exclusive block scan; every thread receives the block total.  smem: >= 32 ints.
__device__ __forceinline__ int block_scan_excl(int v, int* total, int* smem /* >= 32 */) {
  const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
  int x = v;
#pragma unroll
  for (int o = 1; o < 32; o <<= 1) {
    const int y = __shfl_up_sync(0xffffffffu, x, o);
    if (lane >= o) x += y;
  }
  if (lane == 31) smem[wid] = x;
  __syncthreads();
  if (wid == 0) {
    const int nw = blockDim.x >> 5;
    int w = (lane < nw) ? smem[lane] : 0;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
      const int y = __shfl_up_sync(0xffffffffu, w, o);
      if (lane >= o) w += y;
    }
    smem[lane] = w;  // inclusive over warps
  }
  __syncthreads();
  const int base = wid ? smem[wid - 1] : 0;
  *total = smem[(blockDim.x >> 5) - 1];
  __syncthreads();
  return base + x - v;
}

// launchers (one per pipeline step; defined in the .cu of that step)
struct Launch {
  cudaStream_t st;
  int count;          // kernels launched
  cudaEvent_t* kev;   // per-kernel profiling (tpcca_set_profiling(h, 2)): 2 events per timed kernel, or null
};
// Brackets one kernel launch with events when per-kernel profiling is on (id: enum tpcca_kernel_id).
#define KTIMED(L, id, launch)                                   \
  do {                                                          \
    if ((L).kev) cudaEventRecord((L).kev[2 * (id)], (L).st);      \
    launch;                                                     \
    if ((L).kev) cudaEventRecord((L).kev[2 * (id) + 1], (L).st);  \
  } while (0)
cudaError_t setup_grid_kernels();  // per-device function attributes; called by tpcca_init on the handle's device
void launch_grid(const Dev& d, const SecOff& so, Launch& L);
void launch_neighbours(const Dev& d, Launch& L);
void launch_clean_start(const Dev& d, Launch& L);
void launch_tracklets(const Dev& d, Launch& L);
void launch_select(const Dev& d, Launch& L);
void launch_refit(const Dev& d, Launch& L);
void launch_export(const Dev& d, int what, void* dst, Launch& L);
void launch_merge(const Dev& d, Launch& L);
void launch_legs(const Dev& d, Launch& L);
void launch_leg_fit(const Dev& d, Launch& L);
void launch_time_estimate(const Dev& d, float vdrift, float z_max, tpcca_time_rec* out_sector, tpcca_time_rec* out_merged,
                          Launch& L);
// exclusive scan of data[0..n) in place, n read from *n_dev (<= n_max); data[n] receives the total
void launch_scan_i32(int32_t* data, const int32_t* n_dev, int32_t n_max, int32_t* tmp, Launch& L);
// out[0..n) = indices 0..n-1 ordered by decreasing key[i] (keys in [0,256]; order inside a key is arbitrary);
// n read from *n_dev (<= n_max); slot selects the scratch block of Dev::ord
void launch_order_desc(const Dev& d, int slot, const int32_t* key, const int32_t* n_dev, int32_t n_max, int32_t* out,
                       Launch& L);
