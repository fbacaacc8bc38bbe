// tpcca_static.cu -- tpcca_clean_links_static: the link cleaner and start-hit finder (steps (c) and (d) of DESIGN.md,
// PAPER.md:49 "links between hit triplets" kept only when mutual, "concatenates consecutive links" from the chain starts)
// for callers that have no device memory to lend and may not ask the CUDA runtime for any.
//
// Who that is.  Every other entry point of this library works inside a workspace the caller allocated.  Some callers
// cannot do that: a plug-in inside a reconstruction process whose GPU memory was handed over, whole, to the host
// framework's own allocator at start-up (cudaMalloc then fails or is forbidden by policy); a monitoring task that looks
// at the links of a frame another component owns; code in a time-critical loop, where cudaMalloc / cudaFree would
// synchronise the whole device and stall the tracking streams of the neighbouring frames.  For them the compaction
// scratch of this step lives in the library image itself: a file-scope __device__ array of fixed size.  The price is
// stated in include/tpcca.h: a hard size limit, memory held on every GPU that loads the library until the process
// exits, and one array shared by all calls.
//
// Nothing here touches the existing path: tpcca_track keeps using k_clean / k_sb_* in tpcca_links.cu.
#include <cuda_runtime.h>
#include <stdint.h>
#include <stdio.h>

#include <mutex>

#include "../../include/tpcca.h"

void tpcca_internal_set_err(const char* msg);  // tpcca_api.cu: text behind tpcca_last_error() of the calling thread

namespace {

constexpr int CS_THREADS = 256;
constexpr int CS_PER_THREAD = 4;
constexpr int CS_TILE = CS_THREADS * CS_PER_THREAD;  // 1024 clusters per block
constexpr int CS_MAX_TILES = (int)((TPCCA_STATIC_MAX_CLUSTERS + CS_TILE - 1) / CS_TILE);  // 32768
constexpr int CS_HDR = 64;  // int32 words before the per-tile counts (word 0: the ticket counter), keeps the counts 256-byte aligned

// The scratch.  (64 + 32768) * 4 = 131,328 bytes of device memory per GPU, for the life of the process.
//   word 0            ticket counter of the "last block scans" hand-off; MUST be 0 when k_static_clean starts
//   words 64 ...      start hits found in tile b (written by every block), then their exclusive prefix sum (last block)
// In HOST code the name below is only a handle for cudaGetSymbolAddress, never a pointer a kernel could use.
static __device__ __align__(256) int32_t g_static_scratch[CS_HDR + CS_MAX_TILES];

// clean links of cluster h (O3): a link survives only if the partner points back.  Values outside [0, n) count
// as "no link", so a corrupt input can never make the kernel read out of bounds.
__device__ __forceinline__ void clean_one(const int32_t* __restrict__ up, const int32_t* __restrict__ down, int n, int h,
                                          int& u, int& d) {
  u = up[h];
  d = down[h];
  if (u < 0 || u >= n || down[u] != h) u = -1;
  if (d < 0 || d >= n || up[d] != h) d = -1;
}

// inclusive scan over the block's 256 threads; returns the exclusive value, *total = block sum
__device__ __forceinline__ int scan256(int v, int* total, int* sm /* 8 */) {
  const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
  int x = v;
#pragma unroll
  for (int o = 1; o < 32; o <<= 1) {
    const int y = __shfl_up_sync(0xffffffffu, x, o);
    if (lane >= o) x += y;
  }
  if (lane == 31) sm[wid] = x;
  __syncthreads();
  int base = 0, tot = 0;
#pragma unroll
  for (int w = 0; w < CS_THREADS / 32; w++) {
    const int s = sm[w];
    if (w < wid) base += s;
    tot += s;
  }
  __syncthreads();
  *total = tot;
  return base + x - v;
}

// Pass 1: cleaned links out, start hits counted per tile into the scratch; the block that finishes last turns the counts
// into exclusive offsets, writes the total and puts the ticket back to 0 for the next call.
__global__ void __launch_bounds__(CS_THREADS) k_static_clean(const int32_t* __restrict__ up, const int32_t* __restrict__ down,
                                                             int n, int32_t* __restrict__ out_up, int32_t* __restrict__ out_down,
                                                             int32_t* __restrict__ out_n_start, int32_t* scratch) {
  __shared__ int sm[8];
  __shared__ int s_last;
  const int h0 = blockIdx.x * CS_TILE + threadIdx.x * CS_PER_THREAD;
  int mine = 0;
#pragma unroll
  for (int j = 0; j < CS_PER_THREAD; j++) {
    const int h = h0 + j;
    if (h < n) {
      int u, d;
      clean_one(up, down, n, h, u, d);
      out_up[h] = u;
      out_down[h] = d;
      mine += (d < 0 && u >= 0) ? 1 : 0;  // a chain starts here (O4)
    }
  }
  int tot;
  scan256(mine, &tot, sm);
  if (threadIdx.x == 0) {
    scratch[CS_HDR + blockIdx.x] = tot;
    __threadfence();  // the count is visible device-wide before the ticket is taken
    s_last = (atomicAdd(&scratch[0], 1) == (int)gridDim.x - 1) ? 1 : 0;
  }
  __syncthreads();
  if (!s_last) return;
  __threadfence();
  volatile int32_t* cnt = scratch + CS_HDR;  // written by other blocks: read past L1
  int carry = 0;
  for (int b0 = 0; b0 < (int)gridDim.x; b0 += CS_THREADS) {
    const int b = b0 + threadIdx.x;
    const int v = (b < (int)gridDim.x) ? cnt[b] : 0;
    int t;
    const int e = scan256(v, &t, sm);
    if (b < (int)gridDim.x) cnt[b] = carry + e;
    carry += t;
  }
  if (threadIdx.x == 0) {
    *out_n_start = carry;
    scratch[0] = 0;  // ticket ready for the next call
  }
}

// Pass 2: start hits written in ascending cluster index at the tile's offset.  The flags are taken from the cleaned links
// pass 1 wrote (the same decision, and half the reads).
__global__ void __launch_bounds__(CS_THREADS) k_static_starts(const int32_t* __restrict__ cl_up, const int32_t* __restrict__ cl_down,
                                                              int n, int32_t* __restrict__ out_start, const int32_t* __restrict__ scratch) {
  __shared__ int sm[8];
  const int h0 = blockIdx.x * CS_TILE + threadIdx.x * CS_PER_THREAD;
  bool st[CS_PER_THREAD];
  int mine = 0;
#pragma unroll
  for (int j = 0; j < CS_PER_THREAD; j++) {
    const int h = h0 + j;
    st[j] = h < n && cl_down[h] < 0 && cl_up[h] >= 0;
    mine += st[j] ? 1 : 0;
  }
  int tot;
  int pos = scratch[CS_HDR + blockIdx.x] + scan256(mine, &tot, sm);
#pragma unroll
  for (int j = 0; j < CS_PER_THREAD; j++)
    if (st[j]) out_start[pos++] = h0 + j;
}

// Device address of the scratch, looked up once per device with that device current.
constexpr int CS_MAX_DEVICES = 64;
std::mutex g_setup_mutex;
int32_t* g_scratch_addr[CS_MAX_DEVICES];  // zero-initialised: not looked up yet

int fail(int code, const char* msg) {
  tpcca_internal_set_err(msg);
  return code;
}

}  // namespace

extern "C" int tpcca_clean_links_static(const int32_t* link_up_raw, const int32_t* link_down_raw, int64_t n, void* stream,
                                        int32_t* out_link_up, int32_t* out_link_down, int32_t* out_start_hits,
                                        int32_t* out_n_start) {
  char msg[256];
  if (n < 0) return fail(TPCCA_ERR_ARGUMENT, "tpcca_clean_links_static: n is negative");
  if (n > (int64_t)TPCCA_STATIC_MAX_CLUSTERS) {
    snprintf(msg, sizeof(msg),
             "tpcca_clean_links_static: n = %lld exceeds TPCCA_STATIC_MAX_CLUSTERS = %lld (the built-in scratch is fixed; "
             "use tpcca_track with a workspace for larger frames)",
             (long long)n, (long long)TPCCA_STATIC_MAX_CLUSTERS);
    return fail(TPCCA_ERR_ARGUMENT, msg);
  }
  if (!out_n_start || ((uintptr_t)out_n_start & 3)) return fail(TPCCA_ERR_ARGUMENT, "tpcca_clean_links_static: out_n_start null or misaligned");
  if (n > 0 && (!link_up_raw || !link_down_raw || !out_link_up || !out_link_down || !out_start_hits))
    return fail(TPCCA_ERR_ARGUMENT, "tpcca_clean_links_static: null pointer");
  if (((uintptr_t)link_up_raw | (uintptr_t)link_down_raw | (uintptr_t)out_link_up | (uintptr_t)out_link_down |
       (uintptr_t)out_start_hits) & 3)
    return fail(TPCCA_ERR_ARGUMENT, "tpcca_clean_links_static: misaligned pointer (4 B)");
  if (n > 0 && (out_link_up == link_up_raw || out_link_up == link_down_raw || out_link_down == link_up_raw ||
                out_link_down == link_down_raw || out_link_up == out_link_down))
    return fail(TPCCA_ERR_ARGUMENT, "tpcca_clean_links_static: outputs must not alias the inputs or each other");

  int dev = -1;
  cudaError_t e = cudaGetDevice(&dev);
  if (e != cudaSuccess || dev < 0 || dev >= CS_MAX_DEVICES) {
    cudaGetLastError();
    return fail(TPCCA_ERR_CUDA, "tpcca_clean_links_static: no current CUDA device (this library has no CPU fallback)");
  }
  int32_t* scratch;
  {
    // Set-up, first call on this device only: ask the runtime where THIS device keeps its copy of the array.  (The first
    // use of a symbol may make the runtime load the module; that is why the first call belongs outside a stream capture.)
    std::lock_guard<std::mutex> lock(g_setup_mutex);
    if (!g_scratch_addr[dev]) {
      void* p = nullptr;
      e = cudaGetSymbolAddress(&p, g_static_scratch);
      if (e != cudaSuccess || !p) {
        snprintf(msg, sizeof(msg), "tpcca_clean_links_static: cudaGetSymbolAddress failed: %s", cudaGetErrorString(e));
        cudaGetLastError();
        return fail(TPCCA_ERR_CUDA, msg);
      }
      g_scratch_addr[dev] = static_cast<int32_t*>(p);
    }
    scratch = g_scratch_addr[dev];
  }

  cudaStream_t st = (cudaStream_t)stream;
  if (n == 0) {
    e = cudaMemsetAsync(out_n_start, 0, sizeof(int32_t), st);
    if (e != cudaSuccess) { cudaGetLastError(); return fail(TPCCA_ERR_CUDA, "tpcca_clean_links_static: memset failed"); }
    return TPCCA_OK;
  }
  // The array still holds whatever the previous call left.  Only the ticket has to be 0: a completed call leaves it so, a
  // call whose kernel was cut short might not, hence the explicit clear in stream order before every launch.  The counts
  // need no clearing: tile b's word is written by block b before anything reads it.
  e = cudaMemsetAsync(scratch, 0, sizeof(int32_t), st);
  if (e != cudaSuccess) { cudaGetLastError(); return fail(TPCCA_ERR_CUDA, "tpcca_clean_links_static: memset failed"); }
  const int tiles = (int)((n + CS_TILE - 1) / CS_TILE);
  k_static_clean<<<tiles, CS_THREADS, 0, st>>>(link_up_raw, link_down_raw, (int)n, out_link_up, out_link_down, out_n_start, scratch);
  k_static_starts<<<tiles, CS_THREADS, 0, st>>>(out_link_up, out_link_down, (int)n, out_start_hits, scratch);
  e = cudaGetLastError();
  if (e != cudaSuccess) {
    snprintf(msg, sizeof(msg), "tpcca_clean_links_static: kernel launch failed: %s", cudaGetErrorString(e));
    return fail(TPCCA_ERR_CUDA, msg);
  }
  return TPCCA_OK;
}
