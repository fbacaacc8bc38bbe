// tpcca_api.cu -- the C-ABI of include/tpcca.h: argument checks, workspace carving, stream-ordered
// enqueue of steps (a)-(g).  No kernel of the hot path lives here.
#include <math.h>
#include <stdio.h>
#include <stdlib.h>
#include <string.h>

#include <new>

#include "tpcca_dev.cuh"

static thread_local char g_err[512] = "";
static void set_err(const char* fmt, const char* a = "", long long b = 0) { snprintf(g_err, sizeof(g_err), fmt, a, b); }

// for entry points that live in other translation units (tpcca_static.cu)
void tpcca_internal_set_err(const char* msg) { snprintf(g_err, sizeof(g_err), "%s", msg ? msg : ""); }

#define PROF_RING 32
#define MAX_LAYOUT 128
struct tpcca_handle {
  Dev d;
  // workspace layout as carved (offset, bytes used) -- tpcca_debug_workspace_layout
  size_t lay_off[MAX_LAYOUT], lay_bytes[MAX_LAYOUT];
  int n_layout;
  tpcca_geometry geo;
  int64_t max_clusters;
  // host-API staging (inside the workspace): two slots, so that the copies of one frame overlap the kernels of the next
  float4* stage_clusters[2];
  int32_t* stage_assign[2];
  char* stage_tracks[2];
  // pipelined host call (tpcca_track_host_async / tpcca_wait): internal copy streams and per-slot events
  cudaStream_t st_in, st_out, st_rec;
  cudaEvent_t ev_in[2], ev_k[2], ev_out[2];
  struct Pending { bool busy; int64_t n; void* out_tracks; } pend[2];
  // last tpcca_merge (for tpcca_estimate_time and tpcca_find_legs)
  void* last_merged;
  int32_t* last_track_merged;
  int32_t* last_leg_partner;  // out_leg_partner of the last tpcca_find_legs (for tpcca_fit_legs)
  uint64_t seq_submit, seq_wait;
  // Everything above lives in ONE workspace, so the calls on a handle must run on the GPU in the order they were made, also
  // when the caller passes a different stream each time: every entry point that enqueues work first makes its stream wait
  // for ev_last (recorded at the end of the previous one), unless it is the same stream anyway.
  cudaEvent_t ev_last;
  cudaStream_t last_stream;
  bool have_last;
  // last call
  int64_t last_n;
  int launches;
  bool profiling, have_times, debug_sync, kprofiling, have_ktimes;
  cudaEvent_t kev[2 * TPCCA_N_KERNELS];
  int prof_calls;
  int device;
  cudaEvent_t ev[PROF_RING][TPCCA_N_STAGES + 1];
};

static size_t align_up(size_t v) { return (v + 255) & ~(size_t)255; }

// Stream order across calls on one handle (see tpcca_handle::ev_last).
static bool order_after_last(tpcca_handle* h, cudaStream_t st) {
  if (!h->have_last || st == h->last_stream) return true;
  const cudaError_t e = cudaStreamWaitEvent(st, h->ev_last, 0);
  if (e != cudaSuccess) { set_err("cudaStreamWaitEvent failed: %s", cudaGetErrorString(e)); cudaGetLastError(); return false; }
  return true;
}
static void mark_last(tpcca_handle* h, cudaStream_t st) {
  if (cudaEventRecord(h->ev_last, st) == cudaSuccess) { h->last_stream = st; h->have_last = true; }
  else cudaGetLastError();
}

// One pass computes the layout; with base != NULL it also assigns the pointers.
static size_t carve(tpcca_handle* h, const tpcca_geometry* g, const tpcca_params* p, char* base) {
  size_t off = 0;
  const size_t N = (size_t)p->max_clusters, T = (size_t)p->max_tracklets, K = (size_t)p->max_tracks;
  const size_t SL = (size_t)g->n_sectors * g->n_rows;
  const size_t NB = 4 * N + 130 * SL + 2;
  const size_t NSCAN = T + 8 + NB / 2048 + T / 2048 + 64;
  if (base) h->n_layout = 0;
#define CARVE(field, type, count)                                  \
  do {                                                             \
    if (base) {                                                    \
      h->field = reinterpret_cast<type*>(base + off);              \
      if (h->n_layout < MAX_LAYOUT) { h->lay_off[h->n_layout] = off; h->lay_bytes[h->n_layout++] = sizeof(type) * (size_t)(count); } \
    }                                                              \
    off += align_up(sizeof(type) * (size_t)(count));               \
  } while (0)
  CARVE(d.cnt, DevCounters, 1);
  CARVE(d.row_x, const float, g->n_rows);
  CARVE(d.slice_count, int32_t, SL + 1);
  CARVE(d.row_start, int32_t, SL + 1);
  CARVE(d.slice_bbox, uint32_t, SL * 4);
  CARVE(d.grid, GridHdr, SL);
  CARVE(d.nbr, NbrHdr, SL);
  CARVE(d.slice_nstart, int32_t, SL + 1);
  CARVE(d.slice_sbase, int32_t, SL + 1);
  CARVE(d.slice_fill, int32_t, SL + 1);
  CARVE(d.bin_base, int32_t, SL + 1);
  CARVE(d.srec, float4, N);
  CARVE(d.cluster_rank, int32_t, N);
  CARVE(d.bin_start, int32_t, NB + 1);
  CARVE(d.scan_tmp, int32_t, NSCAN);
  CARVE(d.yz, float2, N);
  CARVE(d.orig_idx, int32_t, N);
  CARVE(d.slice_of, uint16_t, N);
  CARVE(d.link_up, int32_t, N);
  CARVE(d.link_down, int32_t, N);
  CARVE(d.link_up_clean, int32_t, N);
  CARVE(d.shared_flag, uint8_t, N);
  CARVE(d.hit_weight, unsigned long long, N);
  CARVE(d.start_tmp, int32_t, N);
  CARVE(d.sb_count, int32_t, T + 1);
  CARVE(d.sb_sorted, int32_t, T);
  CARVE(d.sb_skey, int32_t, T);
  CARVE(d.start_hits, int32_t, T);
  CARVE(d.seed_w, int32_t, T + 1);
  CARVE(d.ord, int32_t, 5 * 1024);
  CARVE(d.e_key, int32_t, 3 * T);
  CARVE(d.e_order, int32_t, 3 * T);
  CARVE(d.work_t, int32_t, T);
  CARVE(d.row_hit, int32_t, T * (size_t)g->n_rows);
  CARVE(d.tl_state, float, T * 40);
  CARVE(d.tl_ints, int32_t, T * 4);
  CARVE(d.tl_floats, float, T * 8);
  CARVE(d.tl_W, unsigned long long, T);
  CARVE(d.sel_scan, int32_t, T + 1);
  CARVE(d.tl_track, int32_t, T + 1);
  CARVE(d.track_tracklet, int32_t, K);
  CARVE(d.track_w, int32_t, K);
  CARVE(d.track_order, int32_t, K);
  CARVE(d.track_len, int32_t, K);
  CARVE(d.w_list, int2, T);
  CARVE(d.th_yz, float2, N);
  CARVE(d.th_row, uint8_t, N);
  CARVE(d.th_hit, int32_t, N);
  CARVE(d.th_shared, uint8_t, N);
  CARVE(d.track_outer, float, K * 24);
  CARVE(d.m_best_out, unsigned long long, K);
  CARVE(d.m_best_in, unsigned long long, K);
  CARVE(d.m_next, int32_t, K);
  CARVE(d.m_prev, int32_t, K);
  CARVE(d.m_scan, int32_t, K + 1);
  CARVE(d.m_head, int32_t, K);
  CARVE(d.m_len, int32_t, K);
  CARVE(d.m_order, int32_t, K);
  CARVE(d.m_cand, int2, K);
  CARVE(d.leg_ends, float4, K * 6);
  CARVE(d.leg_best, unsigned long long, K * 2);
  CARVE(d.leg_sec, int32_t, 2 * (TPCCA_MAX_SECTORS * 128 + 2));   // tpcca_legs.cu: LEG_SEC_STRIDE
  CARVE(d.leg_cur, int32_t, 2 * TPCCA_MAX_SECTORS * 128);
  CARVE(d.leg_list, int32_t, K * 2);
  CARVE(d.leg_bk, float4, K * 4);
  CARVE(d.leg_summary, int32_t, 8);
  for (int sl = 0; sl < 2; sl++) {
    CARVE(stage_clusters[sl], float4, N);
    CARVE(stage_assign[sl], int32_t, N);
    CARVE(stage_tracks[sl], char, sizeof(tpcca_out_header) + K * sizeof(tpcca_track_rec));
  }
#undef CARVE
  if (base) { h->d.max_bins = (int32_t)NB; h->d.sb_key = h->d.cluster_rank; }
  return off;
}

static bool check_geo_params(const tpcca_geometry* g, const tpcca_params* p) {
  if (!g || !p) { set_err("null geometry or params"); return false; }
  if (g->n_sectors < 1 || g->n_sectors > TPCCA_MAX_SECTORS) { set_err("n_sectors out of range [1,64]"); return false; }
  if (g->n_rows < 2 || g->n_rows > TPCCA_MAX_ROWS) { set_err("n_rows out of range [2,256]"); return false; }
  if ((size_t)g->n_sectors * g->n_rows > 65535) { set_err("n_sectors*n_rows must fit 16 bits"); return false; }
  if (p->max_clusters < 0 || p->max_clusters > 400000000LL || p->max_tracklets < 0 || p->max_tracks < 0) {
    set_err("capacities out of range"); return false;
  }
  if (p->min_track_hits < 2 || p->min_tracklet_hits < 2 || p->min_seed_hits < 2) { set_err("min_*_hits must be >= 2"); return false; }
  if (!(p->sigma_y > 0) || !(p->sigma_z > 0)) { set_err("sigma_y/sigma_z must be > 0"); return false; }
  if (!(p->grid_bin_y > 0) || !(p->grid_bin_z_min > 0) || !(p->grid_bins_per_cluster > 0) || p->grid_bins_per_cluster > 4.0f) {
    set_err("grid_* parameters out of range"); return false;
  }
  return true;
}

extern "C" {

void tpcca_default_params(tpcca_params* p) {
  if (!p) return;
  memset(p, 0, sizeof(*p));
  p->sigma_y = 0.1f; p->sigma_z = 0.15f;
  p->nbr_dydx = 1.5f; p->nbr_dzdx = 1.5f; p->nbr_margin_y = 0.5f; p->nbr_margin_z = 0.75f; p->triplet_cut = 18.0f;
  p->cov0[0] = 1.0f; p->cov0[1] = 1.0f; p->cov0[2] = 0.25f; p->cov0[3] = 1.0f; p->cov0[4] = 100.0f;
  p->pick_cut = 16.0f; p->reject_cut = 25.0f; p->max_gap = 5; p->edge_margin = 3.0f; p->max_sinphi = 0.95f;
  p->min_seed_hits = 4; p->min_tracklet_hits = 10; p->min_track_hits = 10; p->qual_scale = 1000.0f;
  p->grid_bin_y = 6.0f; p->grid_bin_z_min = 2.5f; p->grid_bins_per_cluster = 2.0f;
}

void tpcca_default_merge_params(tpcca_merge_params* p) {
  if (!p) return;
  memset(p, 0, sizeof(*p));
  p->merge_chi2_cut = 50.0f; p->merge_dz_max = 30.0f; p->merge_edge_dist = 10.0f;
  p->merge_row_back = 2; p->merge_row_fwd = 8;
  p->fit_reject_cut = 30.0f; p->shared_err_scale = 2.0f; p->ring = 18;
}

size_t tpcca_workspace_bytes(const tpcca_geometry* g, const tpcca_params* p) {
  if (!check_geo_params(g, p)) return 0;
  return carve(nullptr, g, p, nullptr) + 256;
}

tpcca_handle* tpcca_init(const tpcca_geometry* g, float bz_tesla, const tpcca_params* p) {
  if (!check_geo_params(g, p)) return nullptr;
  if (!g->row_x) { set_err("row_x is null"); return nullptr; }
  for (int r = 1; r < g->n_rows; r++)
    if (!(g->row_x[r] > g->row_x[r - 1])) { set_err("row_x must be strictly increasing"); return nullptr; }
  int ndev = 0;
  if (cudaGetDeviceCount(&ndev) != cudaSuccess || ndev == 0) {
    cudaGetLastError();
    set_err("no CUDA device: this library has no CPU fallback");
    return nullptr;
  }
  const size_t need = carve(nullptr, g, p, nullptr) + 256;
  if (!p->workspace || ((uintptr_t)p->workspace & 255) || p->workspace_bytes < need) {
    set_err("workspace null, misaligned (256 B) or too small%s (need %lld bytes)", "", (long long)need);
    return nullptr;
  }
  tpcca_handle* h = new (std::nothrow) tpcca_handle;
  if (!h) { set_err("out of host memory"); return nullptr; }
  memset(h, 0, sizeof(*h));
  h->geo = *g;
  h->geo.row_x = nullptr;
  h->max_clusters = p->max_clusters;
  carve(h, g, p, (char*)p->workspace);
  Dev& d = h->d;
  d.n_sectors = g->n_sectors; d.n_rows = g->n_rows; d.n_slices = g->n_sectors * g->n_rows;
  d.tan_half_angle = g->tan_half_angle;
  d.P = *p;
  d.kq = -((0.000299792458f * 10.0f) * bz_tesla);
  d.sy2 = p->sigma_y * p->sigma_y;
  d.sz2 = p->sigma_z * p->sigma_z;
  d.inv_sy2 = 1.0f / d.sy2;
  d.inv_sz2 = 1.0f / d.sz2;
  d.max_tracklets = p->max_tracklets; d.max_tracks = p->max_tracks;
  if (cudaGetDevice(&h->device) != cudaSuccess ||
      cudaDeviceGetAttribute(&d.n_sm, cudaDevAttrMultiProcessorCount, h->device) != cudaSuccess || d.n_sm < 1) {
    set_err("device query failed: %s", cudaGetErrorString(cudaGetLastError()));
    delete h;
    return nullptr;
  }
  if (setup_grid_kernels() != cudaSuccess) {  // per device: a second device in this process gets its own attribute
    set_err("kernel attribute setup failed: %s", cudaGetErrorString(cudaGetLastError()));
    delete h;
    return nullptr;
  }
  if (cudaMemcpy((void*)d.row_x, g->row_x, sizeof(float) * g->n_rows, cudaMemcpyHostToDevice) != cudaSuccess) {
    set_err("row_x upload failed: %s", cudaGetErrorString(cudaGetLastError()));
    delete h;
    return nullptr;
  }
  for (int k = 0; k < PROF_RING; k++)
    for (int i = 0; i <= TPCCA_N_STAGES; i++)
      if (cudaEventCreate(&h->ev[k][i]) != cudaSuccess) {
        set_err("cudaEventCreate failed: %s", cudaGetErrorString(cudaGetLastError()));
        h->ev[k][i] = nullptr;
        tpcca_free(h);  // destroys the events created so far
        return nullptr;
      }
  bool ok = cudaEventCreateWithFlags(&h->ev_last, cudaEventDisableTiming) == cudaSuccess &&
            cudaStreamCreateWithFlags(&h->st_in, cudaStreamNonBlocking) == cudaSuccess &&
            cudaStreamCreateWithFlags(&h->st_out, cudaStreamNonBlocking) == cudaSuccess &&
            cudaStreamCreateWithFlags(&h->st_rec, cudaStreamNonBlocking) == cudaSuccess;
  for (int sl = 0; sl < 2 && ok; sl++)
    ok = cudaEventCreateWithFlags(&h->ev_in[sl], cudaEventDisableTiming) == cudaSuccess &&
         cudaEventCreateWithFlags(&h->ev_k[sl], cudaEventDisableTiming) == cudaSuccess &&
         cudaEventCreateWithFlags(&h->ev_out[sl], cudaEventDisableTiming) == cudaSuccess;
  if (!ok) {
    set_err("stream / event creation failed: %s", cudaGetErrorString(cudaGetLastError()));
    tpcca_free(h);
    return nullptr;
  }
  return h;
}

static int track_impl(tpcca_handle* h, const tpcca_cluster* clusters, int64_t n, const int32_t* so_host,
                      cudaStream_t st, void* out_tracks, int32_t* out_assign, Launch& L) {
  Dev d = h->d;
  SecOff so;
  memset(&so, 0, sizeof(so));
  if (so_host[0] != 0 || so_host[d.n_sectors] != n) { set_err("sector_offsets must start at 0 and end at n"); return TPCCA_ERR_ARGUMENT; }
  for (int s = 0; s <= d.n_sectors; s++) {
    if (s && so_host[s] < so_host[s - 1]) { set_err("sector_offsets not monotone"); return TPCCA_ERR_ARGUMENT; }
    so.v[s] = so_host[s];
  }
  d.clusters = reinterpret_cast<const float4*>(clusters);
  d.n = (int32_t)n;
  d.out_hdr = reinterpret_cast<tpcca_out_header*>(out_tracks);
  d.out_tracks = reinterpret_cast<tpcca_track_rec*>((char*)out_tracks + sizeof(tpcca_out_header));
  d.out_assign = out_assign;
  h->d.n = d.n; h->d.clusters = d.clusters; h->d.out_hdr = d.out_hdr; h->d.out_tracks = d.out_tracks; h->d.out_assign = out_assign;
  h->last_n = n;
  h->last_merged = nullptr;  // a new frame: the merged tracks of the previous one are gone
  h->last_leg_partner = nullptr;
  const bool prof = h->profiling;
  cudaEvent_t* ev = h->ev[h->prof_calls % PROF_RING];
  // tpcca_set_debug(h, 1): synchronise after every stage and name the stage that faulted (debugging aid)
  const bool dbg = h->debug_sync;
#define DBG_STAGE(name)                                                                          \
  if (dbg) {                                                                                     \
    const cudaError_t de = cudaStreamSynchronize(st);                                            \
    if (de != cudaSuccess) { set_err("stage %s failed: %lld", name, (long long)de); fprintf(stderr, "tpcca: stage %s: %s\n", name, cudaGetErrorString(de)); return TPCCA_ERR_CUDA; } \
  }
  L.kev = (h->kprofiling && h->kev[0]) ? h->kev : nullptr;
  if (prof) cudaEventRecord(ev[0], st);
  launch_grid(d, so, L);
  DBG_STAGE("grid");
  if (prof) cudaEventRecord(ev[1], st);
  launch_neighbours(d, L);
  DBG_STAGE("neighbours");
  if (prof) cudaEventRecord(ev[2], st);
  launch_clean_start(d, L);
  DBG_STAGE("clean_start");
  if (prof) cudaEventRecord(ev[3], st);
  launch_tracklets(d, L);
  DBG_STAGE("tracklets");
  if (prof) cudaEventRecord(ev[4], st);
  launch_select(d, L);
  DBG_STAGE("select");
  if (prof) cudaEventRecord(ev[5], st);
  launch_refit(d, L);
  DBG_STAGE("refit");
#undef DBG_STAGE
  if (prof) cudaEventRecord(ev[6], st);
  if (prof) h->prof_calls++;
  h->have_times = prof && h->prof_calls > 0;
  h->have_ktimes = L.kev != nullptr && d.n > 0 && d.max_tracklets > 0 && d.max_tracks > 0;
  const cudaError_t e = cudaGetLastError();
  if (e != cudaSuccess) { set_err("kernel launch failed: %s", cudaGetErrorString(e)); return TPCCA_ERR_CUDA; }
  return TPCCA_OK;
}

static int check_call(tpcca_handle* h, const void* clusters, int64_t n, const int32_t* so, const void* out_tracks,
                      const void* out_assign) {
  if (!h) { set_err("handle is null (not initialised)"); return TPCCA_ERR_NOT_INIT; }
  if (n < 0 || n > h->max_clusters) { set_err("n out of range%s (max_clusters %lld)", "", (long long)h->max_clusters); return TPCCA_ERR_ARGUMENT; }
  if (!so || !out_tracks) { set_err("sector_offsets or out_tracks is null"); return TPCCA_ERR_ARGUMENT; }
  if (n > 0 && (!clusters || !out_assign)) { set_err("clusters or out_hit_assignment is null"); return TPCCA_ERR_ARGUMENT; }
  if (((uintptr_t)clusters & 15) || ((uintptr_t)out_tracks & 15) || ((uintptr_t)out_assign & 3)) {
    set_err("misaligned pointer (clusters/out_tracks 16 B, assignment 4 B)"); return TPCCA_ERR_ARGUMENT;
  }
  return TPCCA_OK;
}

int tpcca_track(tpcca_handle* h, const tpcca_cluster* clusters, int64_t n, const int32_t* sector_offsets, void* stream,
                void* out_tracks, int32_t* out_hit_assignment) {
  int rc = check_call(h, clusters, n, sector_offsets, out_tracks, out_hit_assignment);
  if (rc) return rc;
  Launch L{(cudaStream_t)stream, 0, nullptr};
  if (!order_after_last(h, L.st)) return TPCCA_ERR_CUDA;
  rc = track_impl(h, clusters, n, sector_offsets, L.st, out_tracks, out_hit_assignment, L);
  h->launches = L.count;
  mark_last(h, L.st);
  return rc;
}

// Pipelined host call.  Frame k uses staging slot k % 2.  Streams: H2D on st_in, kernels on the caller's stream, D2H of
// header + assignment on st_out, D2H of the n_tracks records on st_rec (issued by tpcca_wait once the header is known).
// Events order the three; nothing here blocks the host.
int tpcca_track_host_async(tpcca_handle* h, const tpcca_cluster* clusters, int64_t n, const int32_t* sector_offsets,
                           void* stream, void* out_tracks, int32_t* out_hit_assignment) {
  int rc = check_call(h, clusters, n, sector_offsets, out_tracks, out_hit_assignment);
  if (rc) return rc;
  const int sl = (int)(h->seq_submit & 1);
  if (h->pend[sl].busy) { set_err("two frames are already in flight: call tpcca_wait first"); return TPCCA_ERR_ARGUMENT; }
  cudaStream_t st = (cudaStream_t)stream;
  Launch L{st, 0, nullptr};
  cudaError_t e = cudaSuccess;
  if (n > 0) {
    // the kernels of the frame that used this slot last (two frames ago) read stage_clusters[sl]: they were waited for by
    // tpcca_wait; the event keeps that order explicit.  (Kernel-to-kernel order between frames on different streams is
    // ev_last's job, below.)
    e = cudaStreamWaitEvent(h->st_in, h->ev_k[sl], 0);
    if (e == cudaSuccess) e = cudaMemcpyAsync(h->stage_clusters[sl], clusters, (size_t)n * 16, cudaMemcpyHostToDevice, h->st_in);
  }
  if (e == cudaSuccess) e = cudaEventRecord(h->ev_in[sl], h->st_in);
  if (e == cudaSuccess) e = cudaStreamWaitEvent(st, h->ev_in[sl], 0);
  if (e != cudaSuccess) { set_err("H2D copy failed: %s", cudaGetErrorString(e)); cudaGetLastError(); return TPCCA_ERR_CUDA; }
  // the kernels of this frame reuse the workspace of the previous frame (and of any merge / legs call made on it), which
  // may have been given another stream
  if (!order_after_last(h, st)) return TPCCA_ERR_CUDA;
  rc = track_impl(h, reinterpret_cast<const tpcca_cluster*>(h->stage_clusters[sl]), n, sector_offsets, st,
                  h->stage_tracks[sl], h->stage_assign[sl], L);
  h->launches = L.count;
  mark_last(h, st);
  if (rc) return rc;
  e = cudaEventRecord(h->ev_k[sl], st);
  if (e == cudaSuccess) e = cudaStreamWaitEvent(h->st_out, h->ev_k[sl], 0);
  if (e == cudaSuccess)
    e = cudaMemcpyAsync(out_tracks, h->stage_tracks[sl], sizeof(tpcca_out_header), cudaMemcpyDeviceToHost, h->st_out);
  if (e == cudaSuccess && n > 0)
    e = cudaMemcpyAsync(out_hit_assignment, h->stage_assign[sl], (size_t)n * 4, cudaMemcpyDeviceToHost, h->st_out);
  if (e == cudaSuccess) e = cudaEventRecord(h->ev_out[sl], h->st_out);
  if (e != cudaSuccess) { set_err("D2H enqueue failed: %s", cudaGetErrorString(e)); cudaGetLastError(); return TPCCA_ERR_CUDA; }
  h->pend[sl].busy = true; h->pend[sl].n = n; h->pend[sl].out_tracks = out_tracks;
  h->seq_submit++;
  return TPCCA_OK;
}

// Waits for the OLDEST frame in flight: header and assignment have arrived, then the n_tracks records are copied.
int tpcca_wait(tpcca_handle* h) {
  if (!h) { set_err("handle is null (not initialised)"); return TPCCA_ERR_NOT_INIT; }
  if (h->seq_wait == h->seq_submit) { set_err("no frame in flight"); return TPCCA_ERR_ARGUMENT; }
  const int sl = (int)(h->seq_wait & 1);
  tpcca_handle::Pending& p = h->pend[sl];
  cudaError_t e = cudaEventSynchronize(h->ev_out[sl]);
  if (e == cudaSuccess) {
    const tpcca_out_header* hd = reinterpret_cast<const tpcca_out_header*>(p.out_tracks);
    if (hd->n_tracks > 0) {
      e = cudaMemcpyAsync((char*)p.out_tracks + sizeof(tpcca_out_header), h->stage_tracks[sl] + sizeof(tpcca_out_header),
                          (size_t)hd->n_tracks * sizeof(tpcca_track_rec), cudaMemcpyDeviceToHost, h->st_rec);
      if (e == cudaSuccess) e = cudaStreamSynchronize(h->st_rec);
    }
  }
  p.busy = false;
  h->seq_wait++;
  if (e != cudaSuccess) { set_err("D2H copy / execution failed: %s", cudaGetErrorString(e)); cudaGetLastError(); return TPCCA_ERR_CUDA; }
  return TPCCA_OK;
}

int tpcca_track_host(tpcca_handle* h, const tpcca_cluster* clusters, int64_t n, const int32_t* sector_offsets,
                     void* stream, void* out_tracks, int32_t* out_hit_assignment) {
  if (h && h->seq_wait != h->seq_submit) { set_err("frames of tpcca_track_host_async are in flight: call tpcca_wait first"); return TPCCA_ERR_ARGUMENT; }
  const int rc = tpcca_track_host_async(h, clusters, n, sector_offsets, stream, out_tracks, out_hit_assignment);
  return rc ? rc : tpcca_wait(h);
}

int tpcca_merge(tpcca_handle* h, const tpcca_merge_params* mp, void* stream, void* out_merged, int32_t* out_track_merged) {
  if (!h) { set_err("handle is null (not initialised)"); return TPCCA_ERR_NOT_INIT; }
  if (!mp || !out_merged || !out_track_merged) { set_err("null merge parameters or output"); return TPCCA_ERR_ARGUMENT; }
  if (((uintptr_t)out_merged & 15) || ((uintptr_t)out_track_merged & 3)) { set_err("misaligned merge output"); return TPCCA_ERR_ARGUMENT; }
  if (!h->d.out_hdr) { set_err("tpcca_merge needs a preceding tpcca_track on this handle"); return TPCCA_ERR_ARGUMENT; }
  if (mp->ring < 0 || mp->ring == 1 || mp->ring > TPCCA_MAX_SECTORS || mp->merge_row_back < 0 || mp->merge_row_fwd < 0 ||
      !(mp->shared_err_scale > 0)) {
    set_err("merge parameters out of range (ring must be 0 or 2..64: with ring 1 a sector is its own neighbour)"); return TPCCA_ERR_ARGUMENT;
  }
  Dev d = h->d;
  d.MP = *mp;
  d.merged_hdr = reinterpret_cast<tpcca_out_header*>(out_merged);
  d.merged_out = reinterpret_cast<tpcca_track_rec*>((char*)out_merged + sizeof(tpcca_out_header));
  d.track_merged_out = out_track_merged;
  Launch L{(cudaStream_t)stream, 0, nullptr};
  if (!order_after_last(h, L.st)) return TPCCA_ERR_CUDA;
  launch_merge(d, L);
  mark_last(h, L.st);
  h->launches = L.count;
  h->last_merged = out_merged;
  h->last_track_merged = out_track_merged;
  h->last_leg_partner = nullptr;
  const cudaError_t e = cudaGetLastError();
  if (e != cudaSuccess) { set_err("merge launch failed: %s", cudaGetErrorString(e)); return TPCCA_ERR_CUDA; }
  return TPCCA_OK;
}

void tpcca_default_leg_params(tpcca_leg_params* p) {
  if (!p) return;
  memset(p, 0, sizeof(*p));
  p->leg_min_qpt = 4.0f; p->leg_min_sinphi = 0.5f; p->leg_inner_min_sinphi = 0.2f; p->leg_apex_margin = 2.0f;
  p->leg_max_sector_gap = 5; p->leg_inner_max_sector_gap = 9;
  p->leg_max_turn = 2.9f; p->leg_inner_max_turn = 5.0f; p->leg_centre_frac = 0.05f; p->leg_centre_abs = 1.5f; p->leg_radius_frac = 0.2f;
  p->leg_dz_max = 4.0f; p->leg_dzds_tol = 0.1f;
  p->tag_qpt_low = 20.0f; p->tag_qpt_leg = 5.0f; p->tag_sinphi = 0.8f; p->ring = 18;
}

int tpcca_find_legs(tpcca_handle* h, const tpcca_leg_params* lp, void* stream, int32_t* out_leg_partner,
                    int32_t* out_leg_partner_inner, uint8_t* out_leg_first, uint8_t* out_cluster_tags,
                    tpcca_leg_summary* out_summary) {
  if (!h) { set_err("handle is null (not initialised)"); return TPCCA_ERR_NOT_INIT; }
  if (!lp || !out_leg_partner || !out_leg_partner_inner || !out_leg_first || !out_cluster_tags || !out_summary) { set_err("null leg parameters or output"); return TPCCA_ERR_ARGUMENT; }
  if (((uintptr_t)out_leg_partner & 3) || ((uintptr_t)out_leg_partner_inner & 3) || ((uintptr_t)out_summary & 15)) { set_err("misaligned leg output"); return TPCCA_ERR_ARGUMENT; }
  if (!h->d.out_hdr || !h->last_merged) { set_err("tpcca_find_legs needs a tpcca_merge after the last tpcca_track on this handle"); return TPCCA_ERR_ARGUMENT; }
  if (lp->ring < 0 || lp->ring == 1 || lp->ring > TPCCA_MAX_SECTORS || lp->leg_max_sector_gap < 0 || lp->leg_inner_max_sector_gap < 0 || !(lp->leg_max_turn > 0.0f) ||
      !(lp->leg_max_turn < 3.14159f) || !(lp->leg_inner_max_turn > 0.0f) || !(lp->leg_inner_max_turn < 6.28318f) ||
      !(lp->leg_min_sinphi > 0.0f) || !(lp->leg_inner_min_sinphi > 0.0f) || !(lp->leg_min_qpt > 0.0f) || !(lp->leg_centre_abs >= 0.0f) || !(lp->leg_centre_frac >= 0.0f) ||
      !(lp->leg_centre_abs + lp->leg_centre_frac > 0.0f) || !(lp->leg_radius_frac > 0.0f) || !(lp->leg_dz_max > 0.0f) ||
      !(lp->leg_dzds_tol > 0.0f)) {
    set_err("leg parameters out of range"); return TPCCA_ERR_ARGUMENT;
  }
  Dev d = h->d;
  d.LP = *lp;
  d.merged_out = reinterpret_cast<tpcca_track_rec*>((char*)h->last_merged + sizeof(tpcca_out_header));
  d.track_merged_out = h->last_track_merged;
  d.leg_partner_out = out_leg_partner;
  d.leg_partner_in_out = out_leg_partner_inner;
  d.leg_first_out = out_leg_first;
  d.tags_out = out_cluster_tags;
  d.leg_summary_out = reinterpret_cast<int32_t*>(out_summary);
  Launch L{(cudaStream_t)stream, 0, nullptr};
  if (!order_after_last(h, L.st)) return TPCCA_ERR_CUDA;
  launch_legs(d, L);
  mark_last(h, L.st);
  h->launches = L.count;
  h->last_leg_partner = out_leg_partner;
  const cudaError_t e = cudaGetLastError();
  if (e != cudaSuccess) { set_err("leg launch failed: %s", cudaGetErrorString(e)); return TPCCA_ERR_CUDA; }
  return TPCCA_OK;
}

void tpcca_default_leg_fit_params(tpcca_leg_fit_params* p) {
  if (!p) return;
  memset(p, 0, sizeof(*p));
  p->fit_rot_sinphi = 0.5f; p->fit_step_sinphi = 0.7f; p->fit_min_d = 0.3f; p->fit_reject_cut = 30.0f;
  p->shared_err_scale = 2.0f; p->ring = 18;
}

int tpcca_fit_legs(tpcca_handle* h, const tpcca_leg_fit_params* fp, void* stream, void* out_fits) {
  if (!h) { set_err("handle is null (not initialised)"); return TPCCA_ERR_NOT_INIT; }
  if (!fp || !out_fits) { set_err("null fit parameters or output"); return TPCCA_ERR_ARGUMENT; }
  if ((uintptr_t)out_fits & 15) { set_err("misaligned fit output"); return TPCCA_ERR_ARGUMENT; }
  if (!h->d.out_hdr || !h->last_merged || !h->last_leg_partner) {
    set_err("tpcca_fit_legs needs a tpcca_find_legs after the last tpcca_merge on this handle"); return TPCCA_ERR_ARGUMENT;
  }
  if (fp->ring < 0 || fp->ring > TPCCA_MAX_SECTORS || !(fp->fit_rot_sinphi > 0.0f) || !(fp->fit_rot_sinphi < 0.9f) ||
      !(fp->fit_step_sinphi >= fp->fit_rot_sinphi) || !(fp->fit_step_sinphi < 0.95f) || !(fp->fit_min_d >= 0.0f) ||
      !(fp->shared_err_scale > 0.0f)) {
    set_err("fit parameters out of range"); return TPCCA_ERR_ARGUMENT;
  }
  Dev d = h->d;
  d.FP = *fp;
  d.merged_out = reinterpret_cast<tpcca_track_rec*>((char*)h->last_merged + sizeof(tpcca_out_header));
  d.leg_partner_out = h->last_leg_partner;
  d.fit_hdr = reinterpret_cast<tpcca_out_header*>(out_fits);
  d.fit_out = reinterpret_cast<tpcca_track_rec*>((char*)out_fits + sizeof(tpcca_out_header));
  Launch L{(cudaStream_t)stream, 0, nullptr};
  if (!order_after_last(h, L.st)) return TPCCA_ERR_CUDA;
  launch_leg_fit(d, L);
  mark_last(h, L.st);
  h->launches = L.count;
  const cudaError_t e = cudaGetLastError();
  if (e != cudaSuccess) { set_err("leg fit launch failed: %s", cudaGetErrorString(e)); return TPCCA_ERR_CUDA; }
  return TPCCA_OK;
}

int tpcca_estimate_time(tpcca_handle* h, float vdrift, float z_max, void* stream, tpcca_time_rec* out_sector,
                        tpcca_time_rec* out_merged) {
  if (!h) { set_err("handle is null (not initialised)"); return TPCCA_ERR_NOT_INIT; }
  if (!h->d.out_hdr) { set_err("tpcca_estimate_time needs a preceding tpcca_track on this handle"); return TPCCA_ERR_ARGUMENT; }
  if ((!out_sector && !out_merged) || !(vdrift > 0) || !(z_max > 0)) { set_err("null outputs or bad drift parameters"); return TPCCA_ERR_ARGUMENT; }
  if (((uintptr_t)out_sector & 15) || ((uintptr_t)out_merged & 15)) { set_err("misaligned output"); return TPCCA_ERR_ARGUMENT; }
  if (out_merged && !h->last_merged) { set_err("merged estimates need a tpcca_merge after the last tpcca_track"); return TPCCA_ERR_ARGUMENT; }
  Dev d = h->d;
  if (out_merged) d.merged_out = reinterpret_cast<tpcca_track_rec*>((char*)h->last_merged + sizeof(tpcca_out_header));
  Launch L{(cudaStream_t)stream, 0, nullptr};
  if (!order_after_last(h, L.st)) return TPCCA_ERR_CUDA;
  launch_time_estimate(d, vdrift, z_max, out_sector, out_merged, L);
  mark_last(h, L.st);
  const cudaError_t e = cudaGetLastError();
  if (e != cudaSuccess) { set_err("time estimate launch failed: %s", cudaGetErrorString(e)); return TPCCA_ERR_CUDA; }
  return TPCCA_OK;
}

int tpcca_debug_workspace_layout(tpcca_handle* h, int i, size_t* offset, size_t* bytes) {
  if (!h) { set_err("handle is null (not initialised)"); return TPCCA_ERR_NOT_INIT; }
  if (i < 0 || i >= h->n_layout || !offset || !bytes) return TPCCA_ERR_ARGUMENT;
  *offset = h->lay_off[i];
  *bytes = h->lay_bytes[i];
  return TPCCA_OK;
}

int tpcca_get_intermediate(tpcca_handle* h, int what, void* dst, size_t bytes, void* stream) {
  if (!h) { set_err("handle is null (not initialised)"); return TPCCA_ERR_NOT_INIT; }
  if (!dst || what < 0 || what > TPCCA_MERGE_LINK_NEXT) { set_err("bad intermediate id or null dst"); return TPCCA_ERR_ARGUMENT; }
  if ((uintptr_t)dst & 15) { set_err("dst must be 16-byte aligned"); return TPCCA_ERR_ARGUMENT; }
  const Dev& d = h->d;
  // the sizes of the tracklet / track tables are data dependent: read the live counters (synchronises `stream`;
  // this is a parity / debugging interface, not part of the hot path)
  DevCounters c;
  if (!order_after_last(h, (cudaStream_t)stream)) return TPCCA_ERR_CUDA;
  cudaError_t e = cudaMemcpyAsync(&c, d.cnt, sizeof(c), cudaMemcpyDeviceToHost, (cudaStream_t)stream);
  if (e == cudaSuccess) e = cudaStreamSynchronize((cudaStream_t)stream);
  if (e != cudaSuccess) { set_err("counter copy failed: %s", cudaGetErrorString(e)); cudaGetLastError(); return TPCCA_ERR_CUDA; }
  size_t need;
  if (what <= TPCCA_LINK_DOWN) need = (size_t)d.n * 4;
  else if (what == TPCCA_START_HITS) need = (size_t)c.n_start * 4;
  else if (what == TPCCA_TRACKLET_ROW_HITS) need = (size_t)c.n_start * d.n_rows * 4;
  else if (what == TPCCA_TRACKLET_INTS) need = (size_t)c.n_start * 16;
  else if (what == TPCCA_TRACKLET_FLOATS) need = (size_t)c.n_start * 32;
  else if (what == TPCCA_TRACK_OUTER) need = (size_t)c.n_tracks * 96;
  else if (what == TPCCA_SHARED) need = (size_t)d.n * 4;
  else need = (size_t)c.n_tracks * 4;
  if (bytes < need) { set_err("dst too small%s (need %lld bytes)", "", (long long)need); return TPCCA_ERR_ARGUMENT; }
  Launch L{(cudaStream_t)stream, 0, nullptr};
  launch_export(d, what, dst, L);
  mark_last(h, L.st);
  e = cudaGetLastError();
  if (e != cudaSuccess) { set_err("export launch failed: %s", cudaGetErrorString(e)); return TPCCA_ERR_CUDA; }
  return TPCCA_OK;
}

int tpcca_set_debug(tpcca_handle* h, int on) {
  if (!h) return TPCCA_ERR_NOT_INIT;
  h->debug_sync = on != 0;
  return TPCCA_OK;
}

int tpcca_set_profiling(tpcca_handle* h, int on) {
  if (!h) return TPCCA_ERR_NOT_INIT;
  h->profiling = on != 0;
  h->kprofiling = on >= 2;
  if (on) { h->have_times = false; h->prof_calls = 0; }
  h->have_ktimes = false;
  if (h->kprofiling && !h->kev[0])
    for (int i = 0; i < 2 * TPCCA_N_KERNELS; i++)
      if (cudaEventCreate(&h->kev[i]) != cudaSuccess) {
        // all or nothing: kev[0] != null must mean that every kernel event exists
        cudaGetLastError();
        h->kev[i] = nullptr;
        for (int j = 0; j < i; j++) { cudaEventDestroy(h->kev[j]); h->kev[j] = nullptr; }
        set_err("cudaEventCreate failed"); h->kprofiling = false; return TPCCA_ERR_CUDA;
      }
  return TPCCA_OK;
}

int tpcca_get_kernel_ms(tpcca_handle* h, float* ms) {
  if (!h) return TPCCA_ERR_NOT_INIT;
  if (!ms || !h->have_ktimes) { set_err("no kernel times recorded (tpcca_set_profiling(h, 2) before tpcca_track)"); return TPCCA_ERR_ARGUMENT; }
  for (int i = 0; i < TPCCA_N_KERNELS; i++) {
    if (cudaEventSynchronize(h->kev[2 * i + 1]) != cudaSuccess ||
        cudaEventElapsedTime(&ms[i], h->kev[2 * i], h->kev[2 * i + 1]) != cudaSuccess) {
      set_err("kernel event read failed"); cudaGetLastError(); return TPCCA_ERR_CUDA;
    }
  }
  return TPCCA_OK;
}

int tpcca_get_stage_ms(tpcca_handle* h, float* ms) {
  if (!h) return TPCCA_ERR_NOT_INIT;
  if (!ms || !h->have_times) { set_err("no stage times recorded (enable profiling before tpcca_track)"); return TPCCA_ERR_ARGUMENT; }
  const int nc = h->prof_calls < PROF_RING ? h->prof_calls : PROF_RING;
  for (int i = 0; i < TPCCA_N_STAGES; i++) ms[i] = 0.0f;
  for (int c = 0; c < nc; c++) {
    cudaEvent_t* ev = h->ev[(h->prof_calls - 1 - c) % PROF_RING];
    if (cudaEventSynchronize(ev[TPCCA_N_STAGES]) != cudaSuccess) { set_err("event sync failed"); return TPCCA_ERR_CUDA; }
    for (int i = 0; i < TPCCA_N_STAGES; i++) {
      float t = 0.0f;
      if (cudaEventElapsedTime(&t, ev[i], ev[i + 1]) != cudaSuccess) { set_err("event elapsed failed"); return TPCCA_ERR_CUDA; }
      ms[i] += t / (float)nc;
    }
  }
  return TPCCA_OK;
}

int tpcca_get_stats(tpcca_handle* h, int64_t* stats, void* stream) {
  if (!h) { set_err("handle is null (not initialised)"); return TPCCA_ERR_NOT_INIT; }
  if (!stats) { set_err("stats is null"); return TPCCA_ERR_ARGUMENT; }
  DevCounters c;
  if (!order_after_last(h, (cudaStream_t)stream)) return TPCCA_ERR_CUDA;
  cudaError_t e = cudaMemcpyAsync(&c, h->d.cnt, sizeof(c), cudaMemcpyDeviceToHost, (cudaStream_t)stream);
  if (e == cudaSuccess) e = cudaStreamSynchronize((cudaStream_t)stream);
  if (e != cudaSuccess) { set_err("stats copy failed: %s", cudaGetErrorString(e)); cudaGetLastError(); return TPCCA_ERR_CUDA; }
  stats[TPCCA_WORK_N_BINS] = c.n_bins;
  stats[TPCCA_WORK_ROW_STEPS] = (int64_t)c.row_steps;
  stats[TPCCA_WORK_SEARCHES] = (int64_t)c.searches;
  stats[TPCCA_WORK_TRACK_HITS] = (int64_t)c.track_hits;
  stats[TPCCA_WORK_TRACKLET_HITS] = (int64_t)c.tracklet_hits;
  for (int q = 0; q < 4; q++) stats[TPCCA_WORK_STEPS_E1 + q] = (int64_t)c.phase_steps[q];
  return TPCCA_OK;
}

int tpcca_last_launch_count(tpcca_handle* h) { return h ? h->launches : 0; }

const char* tpcca_last_error(void) { return g_err; }

void tpcca_free(tpcca_handle* h) {
  if (!h) return;
  for (int k = 0; k < PROF_RING; k++)
    for (int i = 0; i <= TPCCA_N_STAGES; i++)
      if (h->ev[k][i]) cudaEventDestroy(h->ev[k][i]);
  for (int sl = 0; sl < 2; sl++) {
    if (h->ev_in[sl]) cudaEventDestroy(h->ev_in[sl]);
    if (h->ev_k[sl]) cudaEventDestroy(h->ev_k[sl]);
    if (h->ev_out[sl]) cudaEventDestroy(h->ev_out[sl]);
  }
  for (int i = 0; i < 2 * TPCCA_N_KERNELS; i++)
    if (h->kev[i]) cudaEventDestroy(h->kev[i]);
  if (h->ev_last) cudaEventDestroy(h->ev_last);
  if (h->st_in) cudaStreamDestroy(h->st_in);
  if (h->st_out) cudaStreamDestroy(h->st_out);
  if (h->st_rec) cudaStreamDestroy(h->st_rec);
  delete h;
}

}  // extern "C"
