/*
 * tpc_synth.c -- seeded synthetic TPC time-frame generator (INPUT GENERATOR ONLY).
 *
 * Serves both the CPU oracle and the CUDA path with identical input bytes.  It holds
 * none of the tracking method's arithmetic: it only draws helices and turns them into
 * clusters, in float64, rounding once to fp32 at the end.  Recipe: DESIGN.md "Input
 * recipe" (BASELINE.json configs 1-5; PAPER.md:41 152 pad rows; PAPER.md:49 36 sectors;
 * PAPER.md:93 cluster time scaled linearly to z, "arbitrarily long TPC").
 *
 * Random numbers: counter-based (splitmix64 finaliser over (seed, stream, counter)), so
 * every track owns its stream and the output does not depend on evaluation order.
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>

typedef struct {
  int32_t n_sectors;      /* 1 (config 1: one standalone sector) or 36 */
  int32_t n_rows;         /* 152 */
  double x_first, x_last; /* 85, 245 cm, rows linearly spaced */
  double bz_tesla;        /* 0.5 */
  uint64_t seed;
  int32_t n_collisions;
  int32_t mult_lo, mult_hi, mult_log_uniform; /* primaries per collision */
  int32_t pt_law;         /* 0 log-uniform [pt_lo,pt_hi]; 1 exponential(mean) truncated */
  double pt_lo, pt_hi, pt_mean;
  double eta_max;
  double vz_sigma;        /* vertex z ~ N(0, vz_sigma) */
  int32_t phi_in_sector;  /* 1: phi uniform inside the +-10 deg of the single sector */
  int32_t n_loopers;      /* extra low-pT helices per collision */
  double looper_pt_lo, looper_pt_hi;
  double time_window_us;  /* collision time uniform in [0, window) */
  double vdrift;          /* cm/us */
  double sigma_y, sigma_z;
  double noise_frac;
  double z_max;           /* drift length, 250 cm */
  int32_t max_turns;      /* 10 */
} synth_config;

typedef struct {
  int64_t n;              /* clusters */
  int32_t n_tracks;
  float *xyz;             /* n*3 */
  int32_t *row;           /* n */
  int32_t *truth;         /* n: generator track id or -1 (noise) */
  int32_t *sector_offsets;/* n_sectors+1 */
  double *track_par;      /* n_tracks*8: pt, phi0, eta, charge, vz, t0_us, collision, n_clusters */
} synth_frame;

/* ---- counter-based RNG ---- */
static uint64_t mix64(uint64_t z) {
  z += 0x9E3779B97F4A7C15ULL;
  z = (z ^ (z >> 30)) * 0xBF58476D1CE4E5B9ULL;
  z = (z ^ (z >> 27)) * 0x94D049BB133111EBULL;
  return z ^ (z >> 31);
}
typedef struct { uint64_t key, ctr; } rng_t;
static rng_t rng_make(uint64_t seed, uint64_t stream) {
  rng_t r; r.key = mix64(mix64(seed) ^ (stream * 0xD1342543DE82EF95ULL)); r.ctr = 0; return r;
}
static uint64_t rng_u64(rng_t *r) { return mix64(r->key + (r->ctr++) * 0x9E3779B97F4A7C15ULL); }
static double rng_uniform(rng_t *r) { return ((double)(rng_u64(r) >> 11) + 0.5) * (1.0 / 9007199254740992.0); }
static double rng_normal(rng_t *r) { /* Box-Muller */
  double u1 = rng_uniform(r), u2 = rng_uniform(r);
  return sqrt(-2.0 * log(u1)) * cos(6.283185307179586476925 * u2);
}

/* ---- growable cluster buffer ---- */
typedef struct { double y, z; int32_t row, sector, truth; } gcl;
typedef struct { gcl *p; int64_t n, cap; } gbuf;
static int gpush(gbuf *b, gcl c) {
  if (b->n == b->cap) {
    int64_t nc = b->cap ? b->cap * 2 : (1 << 16);
    gcl *q = (gcl *)realloc(b->p, (size_t)nc * sizeof(gcl));
    if (!q) return -1;
    b->p = q; b->cap = nc;
  }
  b->p[b->n++] = c; return 0;
}

#define PI 3.14159265358979323846

/* One helix from (0,0,vz): clusters on every pad-row crossing in every sector. */
static int trace_helix(const synth_config *c, gbuf *out, rng_t *rng, int32_t tid, double pt, double phi0,
                       double eta, double q, double vz, double t0, int32_t *n_made) {
  const int nsec_phi = (c->n_sectors == 1) ? 1 : 18;
  const double kappa = -0.00299792458 * c->bz_tesla * q / pt; /* dpsi/ds, 1/cm */
  const double tl = sinh(eta);
  const double tan_half = tan(10.0 * PI / 180.0);
  const double turn_len = 2.0 * PI / fabs(kappa);
  const double dxrow = (c->x_last - c->x_first) / (double)(c->n_rows - 1);
  int32_t made = 0;
  for (int k = 0; k < nsec_phi; k++) {
    const double alpha = (c->n_sectors == 1) ? 0.0 : (20.0 * k + 10.0) * PI / 180.0;
    const double psi0 = phi0 - alpha;
    const double s0 = sin(psi0), c0 = cos(psi0);
    for (int r = 0; r < c->n_rows; r++) {
      const double xr = c->x_first + dxrow * r;
      const double S = s0 + kappa * xr; /* sin(psi_local) is linear in local x */
      if (!(fabs(S) < 1.0)) continue;
      const double cabs = sqrt(1.0 - S * S);
      for (int root = 0; root < 2; root++) {
        const double cr = root ? -cabs : cabs;        /* outgoing / returning */
        const double yl = -(cr - c0) / kappa;
        if (fabs(yl) > xr * tan_half) continue;
        const double psi = atan2(S, cr);
        double dpsi = (psi - psi0) * (kappa > 0 ? 1.0 : -1.0); /* turning angle, >= 0 */
        dpsi = fmod(dpsi, 2.0 * PI);
        if (dpsi < 0) dpsi += 2.0 * PI;
        const double sbase = dpsi / fabs(kappa);
        for (int turn = 0; turn < c->max_turns; turn++) {
          const double s = sbase + turn * turn_len;
          double z = vz + s * tl;
          if (fabs(z) > c->z_max) continue;
          gcl g;
          g.row = r;
          g.y = yl + c->sigma_y * rng_normal(rng);
          z += c->sigma_z * rng_normal(rng);
          const int side = (z < 0.0) ? 1 : 0;
          g.z = z + (side ? -1.0 : 1.0) * c->vdrift * t0; /* PAPER.md:93 time -> z */
          g.sector = (c->n_sectors == 1) ? 0 : k + 18 * side;
          g.truth = tid;
          if (gpush(out, g)) return -1;
          made++;
        }
      }
    }
  }
  *n_made = made;
  return 0;
}

static int cmp_sector(const void *a, const void *b) {
  const gcl *x = (const gcl *)a, *y = (const gcl *)b;
  return (x->sector > y->sector) - (x->sector < y->sector);
}

void synth_free(synth_frame *f) {
  if (!f) return;
  free(f->xyz); free(f->row); free(f->truth); free(f->sector_offsets); free(f->track_par); free(f);
}

synth_frame *synth_generate(const synth_config *c) {
  gbuf buf = {0, 0, 0};
  synth_frame *f = (synth_frame *)calloc(1, sizeof(synth_frame));
  if (!f) return 0;
  /* pass 1: multiplicities */
  int32_t *mult = (int32_t *)malloc(sizeof(int32_t) * (size_t)c->n_collisions);
  double *tcol = (double *)malloc(sizeof(double) * (size_t)c->n_collisions);
  int64_t ntr = 0;
  for (int ic = 0; ic < c->n_collisions; ic++) {
    rng_t r = rng_make(c->seed, 0x1000000ULL + (uint64_t)ic);
    int32_t m = c->mult_lo;
    if (c->mult_log_uniform) {
      double u = rng_uniform(&r);
      m = (int32_t)floor(exp(log((double)c->mult_lo) + u * (log((double)c->mult_hi) - log((double)c->mult_lo))) + 0.5);
    }
    mult[ic] = m + c->n_loopers;
    tcol[ic] = (c->time_window_us > 0) ? rng_uniform(&r) * c->time_window_us : 0.0;
    ntr += mult[ic];
  }
  f->n_tracks = (int32_t)ntr;
  f->track_par = (double *)calloc((size_t)ntr * 8 + 1, sizeof(double));
  int32_t tid = 0;
  for (int ic = 0; ic < c->n_collisions; ic++) {
    rng_t rc = rng_make(c->seed, 0x2000000ULL + (uint64_t)ic);
    const double vz = c->vz_sigma > 0 ? c->vz_sigma * rng_normal(&rc) : 0.0;
    for (int it = 0; it < mult[ic]; it++, tid++) {
      rng_t r = rng_make(c->seed, 0x100000000ULL + (uint64_t)tid);
      const int looper = it >= mult[ic] - c->n_loopers;
      double pt;
      if (looper) {
        pt = c->looper_pt_lo + rng_uniform(&r) * (c->looper_pt_hi - c->looper_pt_lo);
      } else if (c->pt_law == 0) {
        pt = exp(log(c->pt_lo) + rng_uniform(&r) * (log(c->pt_hi) - log(c->pt_lo)));
      } else { /* exponential with mean pt_mean, truncated to [pt_lo, pt_hi]: inverse CDF */
        const double a = exp(-c->pt_lo / c->pt_mean), b = exp(-c->pt_hi / c->pt_mean);
        pt = -c->pt_mean * log(a - rng_uniform(&r) * (a - b));
      }
      double phi0 = c->phi_in_sector ? (rng_uniform(&r) * 2.0 - 1.0) * (10.0 * PI / 180.0)
                                     : rng_uniform(&r) * 2.0 * PI;
      const double eta = (rng_uniform(&r) * 2.0 - 1.0) * c->eta_max;
      const double q = rng_uniform(&r) < 0.5 ? -1.0 : 1.0;
      int32_t made = 0;
      if (trace_helix(c, &buf, &r, tid, pt, phi0, eta, q, vz, tcol[ic], &made)) { synth_free(f); free(buf.p); return 0; }
      double *tp = f->track_par + (size_t)tid * 8;
      tp[0] = pt; tp[1] = phi0; tp[2] = eta; tp[3] = q; tp[4] = vz; tp[5] = tcol[ic]; tp[6] = ic; tp[7] = made;
    }
  }
  free(mult); free(tcol);
  /* noise: ceil(frac * signal) per sector; row uniform, y uniform in the row, z uniform over the side's span */
  const int ns = c->n_sectors;
  int64_t *cnt = (int64_t *)calloc((size_t)ns + 1, sizeof(int64_t));
  for (int64_t i = 0; i < buf.n; i++) cnt[buf.p[i].sector]++;
  const double zspan = c->z_max + c->vdrift * c->time_window_us;
  const double dxrow = (c->x_last - c->x_first) / (double)(c->n_rows - 1);
  const double tan_half = tan(10.0 * PI / 180.0);
  for (int s = 0; s < ns; s++) {
    const int64_t nn = (int64_t)ceil(c->noise_frac * (double)cnt[s]);
    rng_t r = rng_make(c->seed, 0x3000000ULL + (uint64_t)s);
    for (int64_t i = 0; i < nn; i++) {
      gcl g;
      g.row = (int32_t)(rng_uniform(&r) * c->n_rows);
      if (g.row >= c->n_rows) g.row = c->n_rows - 1;
      const double xr = c->x_first + dxrow * g.row;
      g.y = (rng_uniform(&r) * 2.0 - 1.0) * xr * tan_half;
      double z = rng_uniform(&r) * zspan;
      if (ns == 1) z = (rng_uniform(&r) * 2.0 - 1.0) * zspan; /* standalone sector: both signs */
      else if (s >= 18) z = -z;
      g.z = z; g.sector = s; g.truth = -1;
      if (gpush(&buf, g)) { synth_free(f); free(buf.p); free(cnt); return 0; }
    }
  }
  free(cnt);
  /* group by sector (stable w.r.t. nothing: the shuffle below fixes the order) */
  qsort(buf.p, (size_t)buf.n, sizeof(gcl), cmp_sector);
  f->n = buf.n;
  f->sector_offsets = (int32_t *)calloc((size_t)ns + 1, sizeof(int32_t));
  for (int64_t i = 0; i < buf.n; i++) f->sector_offsets[buf.p[i].sector + 1]++;
  for (int s = 0; s < ns; s++) f->sector_offsets[s + 1] += f->sector_offsets[s];
  /* qsort is not stable: make the pre-shuffle order canonical (truth, row, z, y) inside a sector by
     shuffling with keys that do not depend on it -- sort by a hash of the cluster's own content. */
  for (int s = 0; s < ns; s++) {
    const int64_t b = f->sector_offsets[s], e = f->sector_offsets[s + 1];
    /* content-keyed shuffle: key = mix(seed, bits(y), bits(z), row, truth); sort by key */
    uint64_t *key = (uint64_t *)malloc(sizeof(uint64_t) * (size_t)(e - b + 1));
    int64_t *idx = (int64_t *)malloc(sizeof(int64_t) * (size_t)(e - b + 1));
    for (int64_t i = b; i < e; i++) {
      uint64_t by, bz; memcpy(&by, &buf.p[i].y, 8); memcpy(&bz, &buf.p[i].z, 8);
      key[i - b] = mix64(mix64(mix64(c->seed ^ by) ^ bz) ^ ((uint64_t)(uint32_t)buf.p[i].row << 32 | (uint32_t)buf.p[i].truth));
      idx[i - b] = i;
    }
    /* simple LSD radix sort on 64-bit keys, 8 passes */
    const int64_t m = e - b;
    uint64_t *k2 = (uint64_t *)malloc(sizeof(uint64_t) * (size_t)(m + 1));
    int64_t *i2 = (int64_t *)malloc(sizeof(int64_t) * (size_t)(m + 1));
    for (int pass = 0; pass < 8; pass++) {
      int64_t h[257]; memset(h, 0, sizeof(h));
      for (int64_t i = 0; i < m; i++) h[((key[i] >> (8 * pass)) & 255) + 1]++;
      for (int j = 0; j < 256; j++) h[j + 1] += h[j];
      for (int64_t i = 0; i < m; i++) { int64_t d = h[(key[i] >> (8 * pass)) & 255]++; k2[d] = key[i]; i2[d] = idx[i]; }
      uint64_t *tk = key; key = k2; k2 = tk; int64_t *ti = idx; idx = i2; i2 = ti;
    }
    gcl *tmp = (gcl *)malloc(sizeof(gcl) * (size_t)(m + 1));
    for (int64_t i = 0; i < m; i++) tmp[i] = buf.p[idx[i]];
    memcpy(buf.p + b, tmp, sizeof(gcl) * (size_t)m);
    free(tmp); free(key); free(idx); free(k2); free(i2);
  }
  f->xyz = (float *)malloc(sizeof(float) * 3 * (size_t)(buf.n + 1));
  f->row = (int32_t *)malloc(sizeof(int32_t) * (size_t)(buf.n + 1));
  f->truth = (int32_t *)malloc(sizeof(int32_t) * (size_t)(buf.n + 1));
  for (int64_t i = 0; i < buf.n; i++) {
    const gcl *g = &buf.p[i];
    f->xyz[3 * i + 0] = (float)(c->x_first + dxrow * g->row);
    f->xyz[3 * i + 1] = (float)g->y;
    f->xyz[3 * i + 2] = (float)g->z;
    f->row[i] = g->row;
    f->truth[i] = g->truth;
  }
  free(buf.p);
  return f;
}

int64_t synth_n(const synth_frame *f) { return f->n; }
int32_t synth_n_tracks(const synth_frame *f) { return f->n_tracks; }
const float *synth_xyz(const synth_frame *f) { return f->xyz; }
const int32_t *synth_row(const synth_frame *f) { return f->row; }
const int32_t *synth_truth(const synth_frame *f) { return f->truth; }
const int32_t *synth_sector_offsets(const synth_frame *f) { return f->sector_offsets; }
const double *synth_track_par(const synth_frame *f) { return f->track_par; }
