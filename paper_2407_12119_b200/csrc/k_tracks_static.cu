// etx_tracks_static: the track-container regrouping of etx_tracks (include/etx.h) for callers
// that must not allocate device memory.
//
// Who that is.  The paper's pipeline is meant to run inside Allen, LHCb's GPU trigger framework: there
// every algorithm receives its buffers from a per-stream arena that the framework sized up front, and nothing inside
// the event loop may call cudaMalloc / cudaFree -- those calls take a device-wide lock and can wait for every stream
// to drain, which stalls the other streams of events that are in flight.  The same holds for a plug-in that is handed
// nothing but raw device pointers by a host application that owns all of the device memory and gives out no allocator.
// etx_tracks needs a handle, and a handle is created by allocating its workspace; this entry point needs no handle.
//
// How.  The four per-hit work arrays and the block sums of the two prefix sums live in ONE file-scope __device__ array
// of fixed size, part of the library image: each GPU that loads libetx.so holds kScratchBytes (about 16 MiB) of it from
// the moment the library's module is loaded on that GPU until the process exits, whether or not this call is ever made.
// The caller passes inputs and outputs; the call issues kernel launches and cudaMemsetAsync on the caller's stream and
// nothing else -- no cudaMalloc, no cudaFree, no cudaHostAlloc, no library routine that allocates.
//
// Consequences the caller has to know (they are repeated in include/etx.h):
//   * n_hits above ETX_TRACKS_STATIC_MAX_HITS is refused with ETX_ERR_CAPACITY; nothing is launched.
//   * The first call on a device looks up the device address of the array (cudaGetSymbolAddress, once per device,
//     with that device current).  That lookup may load the module, so make the first call on every device before any
//     stream capture begins.
//   * All calls on one GPU share the one array, and it still holds what the previous call left there.  The call clears
//     the two arrays that must start at zero itself.  Two calls whose work overlaps in time on the same GPU (different
//     streams, or different host threads) corrupt each other: order them, on one stream or with events.
//
// The arithmetic is the one of launch_tracks in k_graph.cu (integer work, so the results are equal bit for bit);
// the kernels here are this file's own so that the existing path is untouched.
#include <cuda_runtime.h>
#include <stdint.h>
#include <stdio.h>

#include <mutex>

#include "../../include/etx.h"

namespace {

constexpr int kMaxHits = ETX_TRACKS_STATIC_MAX_HITS;
constexpr int kThreads = 256;
constexpr int kItems = 8;                                  // prefix sum: consecutive elements per thread
constexpr int kChunk = kThreads * kItems;                  // ... and per block
constexpr int kMaxBlocks = (kMaxHits + kChunk - 1) / kChunk;
static_assert(kMaxBlocks <= 1024, "the block sums are scanned by one block, one element per thread");

// Layout of the scratch array, in int32 elements.  Every part starts on a 256-byte boundary.
constexpr size_t kOffSize = 0;                             // [n]      hits per component, indexed by root
constexpr size_t kOffKeep = kOffSize + kMaxHits;           // [n]      1 iff root of a kept track; later the fill cursors
constexpr size_t kOffKsize = kOffKeep + kMaxHits;          // [n]      sizes of the kept tracks in dense order
constexpr size_t kOffNumber = kOffKsize + kMaxHits;        // [n + 1]  dense number of every root (prefix sum of keep)
constexpr size_t kOffBsum = kOffNumber + kMaxHits + 64;    // [blocks] block sums of the running prefix sum
constexpr size_t kScratchInts = kOffBsum + 1024;
constexpr size_t kScratchBytes = kScratchInts * sizeof(int32_t);

// The scratch memory itself.  In HOST code this name is only a handle for the runtime's symbol table -- it is not a
// device address and must never be passed to a kernel; scratch_for_current_device() below asks the runtime for the
// real address.  (Device code could name it directly; the kernels take pointers so that they read like the originals.)
static __device__ __align__(256) int32_t g_tracks_scratch[kScratchInts];

constexpr int kMaxDevices = 64;
int32_t* g_scratch_addr[kMaxDevices] = {};                 // device address of g_tracks_scratch on device i, once known
std::mutex g_setup_mutex;
thread_local char g_error[256] = "";

etx_status fail(etx_status st, const char* what, cudaError_t e = cudaSuccess) {
  if (e != cudaSuccess) snprintf(g_error, sizeof g_error, "etx_tracks_static: %s: %s", what, cudaGetErrorString(e));
  else snprintf(g_error, sizeof g_error, "etx_tracks_static: %s", what);
  return st;
}

// Once per device, with that device current: the address of this device's copy of the array.
etx_status scratch_for_current_device(int32_t** out) {
  int dev = -1;
  cudaError_t e = cudaGetDevice(&dev);
  if (e != cudaSuccess) return fail(ETX_ERR_CUDA, "cudaGetDevice", e);
  if (dev < 0 || dev >= kMaxDevices) return fail(ETX_ERR_UNSUPPORTED, "device ordinal beyond 63");
  std::lock_guard<std::mutex> lock(g_setup_mutex);
  if (!g_scratch_addr[dev]) {
    void* p = nullptr;
    e = cudaGetSymbolAddress(&p, g_tracks_scratch);
    if (e != cudaSuccess || !p) return fail(ETX_ERR_CUDA, "cudaGetSymbolAddress(scratch)", e);
    g_scratch_addr[dev] = static_cast<int32_t*>(p);
  }
  *out = g_scratch_addr[dev];
  return ETX_OK;
}

// ---- prefix sum: out[0..n] = exclusive sums of in[0..n), optionally *total = out[n] ---------------------------------
__device__ __forceinline__ int block_exclusive(int v, int* block_total) {      // blockDim.x == kThreads
  __shared__ int wsum[kThreads / 32];
  const int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
  int incl = v;
#pragma unroll
  for (int o = 1; o < 32; o <<= 1) { const int y = __shfl_up_sync(0xffffffffu, incl, o); if (lane >= o) incl += y; }
  if (lane == 31) wsum[w] = incl;
  __syncthreads();
  int before = 0, all = 0;
#pragma unroll
  for (int i = 0; i < kThreads / 32; ++i) { const int s = wsum[i]; if (i < w) before += s; all += s; }
  __syncthreads();                                                              // wsum is reused by the next call
  *block_total = all;
  return before + incl - v;
}

__global__ void __launch_bounds__(kThreads) st_block_sums_kernel(const int32_t* __restrict__ in, int n, int32_t* __restrict__ bsum) {
  const int first = blockIdx.x * kChunk + threadIdx.x * kItems;
  int v = 0;
#pragma unroll
  for (int j = 0; j < kItems; ++j) if (first + j < n) v += in[first + j];
  int tot;
  block_exclusive(v, &tot);
  if (threadIdx.x == 0) bsum[blockIdx.x] = tot;
}

__global__ void __launch_bounds__(1024) st_scan_block_sums_kernel(int32_t* __restrict__ bsum, int nb) {   // one block, nb <= 1024
  __shared__ int part[32];
  const int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
  const int v = (int)threadIdx.x < nb ? bsum[threadIdx.x] : 0;
  int incl = v;
#pragma unroll
  for (int o = 1; o < 32; o <<= 1) { const int y = __shfl_up_sync(0xffffffffu, incl, o); if (lane >= o) incl += y; }
  if (lane == 31) part[w] = incl;
  __syncthreads();
  int before = 0;
  for (int i = 0; i < w; ++i) before += part[i];
  if ((int)threadIdx.x < nb) bsum[threadIdx.x] = before + incl - v;
}

__global__ void __launch_bounds__(kThreads) st_scan_write_kernel(const int32_t* __restrict__ in, int n, const int32_t* __restrict__ bsum,
                                                                 int32_t* __restrict__ out, int32_t* __restrict__ total) {
  const int first = blockIdx.x * kChunk + threadIdx.x * kItems;
  int x[kItems], v = 0;
#pragma unroll
  for (int j = 0; j < kItems; ++j) { x[j] = first + j < n ? in[first + j] : 0; v += x[j]; }
  int tot;
  int run = block_exclusive(v, &tot) + bsum[blockIdx.x];
#pragma unroll
  for (int j = 0; j < kItems; ++j) {
    const int i = first + j;
    if (i < n) out[i] = run;
    run += x[j];
    if (i == n - 1) { out[n] = run; if (total) *total = run; }
  }
}

void exclusive_scan(const int32_t* in, int n, int32_t* out, int32_t* total, int32_t* bsum, cudaStream_t s) {   // n >= 1
  const int nb = (n + kChunk - 1) / kChunk;
  st_block_sums_kernel<<<nb, kThreads, 0, s>>>(in, n, bsum);
  st_scan_block_sums_kernel<<<1, 1024, 0, s>>>(bsum, nb);
  st_scan_write_kernel<<<nb, kThreads, 0, s>>>(in, n, bsum, out, total);
}

// ---- regrouping (the steps of launch_tracks, k_graph.cu) ------------------------------------------------------------
// A track id outside [0, n) cannot come out of etx_run; it is skipped here so that a foreign input cannot make these
// kernels write outside the scratch array.
__global__ void st_size_kernel(const int32_t* __restrict__ track_id, int n, int32_t* __restrict__ size) {
  const int h = blockIdx.x * blockDim.x + threadIdx.x;
  if (h >= n) return;
  const unsigned r = (unsigned)track_id[h];
  if (r < (unsigned)n) atomicAdd(&size[r], 1);
}
__global__ void st_keep_kernel(const int32_t* __restrict__ track_id, const int32_t* __restrict__ size, int n, int min_hits,
                               int32_t* __restrict__ keep) {
  const int r = blockIdx.x * blockDim.x + threadIdx.x;
  if (r < n) keep[r] = (track_id[r] == r && size[r] >= min_hits) ? 1 : 0;
}
__global__ void st_index_kernel(const int32_t* __restrict__ track_id, const int32_t* __restrict__ size,
                                const int32_t* __restrict__ number, int n, int min_hits,
                                int32_t* __restrict__ track_index, int32_t* __restrict__ ksize) {
  const int h = blockIdx.x * blockDim.x + threadIdx.x;
  if (h >= n) return;
  const unsigned r = (unsigned)track_id[h];
  const bool kept = r < (unsigned)n && size[r] >= min_hits;
  track_index[h] = kept ? number[r] : -1;
  if (kept && (int)r == h) ksize[number[r]] = size[r];
}
__global__ void st_event_kernel(const int32_t* __restrict__ event_off, const int32_t* __restrict__ number, int n_events, int n,
                                int32_t* __restrict__ event_track_off) {
  const int e = blockIdx.x * blockDim.x + threadIdx.x;
  if (e <= n_events) event_track_off[e] = number[min(max(event_off[e], 0), n)];
}
// One warp per event, 32 hits per step in ascending order; lanes with the same track are ranked among themselves and
// the lowest of them moves the track's cursor, so each hit list ascends.  Only this warp touches its event's cursors.
__global__ void __launch_bounds__(256)
st_fill_kernel(const int32_t* __restrict__ track_index, const int32_t* __restrict__ track_offsets,
               const int32_t* __restrict__ event_off, const int32_t* __restrict__ event_track_off, int n_events, int n,
               int32_t* cursor, int32_t* __restrict__ track_hits) {
  const int e = blockIdx.x * 8 + (threadIdx.x >> 5), lane = threadIdx.x & 31;
  if (e >= n_events) return;
  const int h0 = max(event_off[e], 0), h1 = min(event_off[e + 1], n);
  const int t0 = event_track_off[e], t1 = event_track_off[e + 1];
  volatile int32_t* cur = cursor;
  for (int t = t0 + lane; t < t1; t += 32) cur[t] = track_offsets[t];
  __syncwarp();
  for (int i0 = h0; i0 < h1; i0 += 32) {
    const int h = i0 + lane;
    const int t = h < h1 ? track_index[h] : -1;
    const unsigned active = __ballot_sync(0xffffffffu, t >= 0);
    if (t >= 0) {
      const unsigned peers = __match_any_sync(active, t);
      const int leader = __ffs(peers) - 1, rank = __popc(peers & ((1u << lane) - 1u));
      int pos = 0;
      if (lane == leader) { pos = cur[t]; cur[t] = pos + __popc(peers); }
      pos = __shfl_sync(peers, pos, leader);
      track_hits[pos + rank] = h;
    }
    __syncwarp();
  }
}

}  // namespace

extern "C" etx_status etx_tracks_static(const int32_t* d_track_id, const int32_t* d_event_offsets, int32_t n_hits,
                                        int32_t n_events, int32_t min_hits, etx_stream stream, int32_t* d_track_index,
                                        int32_t* d_track_offsets, int32_t* d_track_hits, int32_t* d_event_track_offsets,
                                        int32_t* d_n_tracks) {
  g_error[0] = 0;
  if (n_hits < 0 || n_events < 0 || min_hits < 1) return fail(ETX_ERR_ARG, "negative size or min_hits < 1");
  if (!d_event_offsets || !d_track_offsets || !d_event_track_offsets || !d_n_tracks)
    return fail(ETX_ERR_ARG, "null offsets / count pointer");
  if (n_hits > 0 && (!d_track_id || !d_track_index || !d_track_hits)) return fail(ETX_ERR_ARG, "null per-hit pointer");
  if (n_hits > kMaxHits) {
    snprintf(g_error, sizeof g_error, "etx_tracks_static: n_hits = %d exceeds ETX_TRACKS_STATIC_MAX_HITS = %d (the fixed scratch array); "
             "split the batch at an event boundary or use etx_tracks", n_hits, kMaxHits);
    return ETX_ERR_CAPACITY;
  }
  int32_t* scratch = nullptr;
  const etx_status st = scratch_for_current_device(&scratch);
  if (st != ETX_OK) return st;
  cudaStream_t s = static_cast<cudaStream_t>(stream);

  cudaMemsetAsync(d_n_tracks, 0, sizeof(int32_t), s);
  if (n_hits == 0 || n_events == 0) {
    cudaMemsetAsync(d_event_track_offsets, 0, sizeof(int32_t) * ((size_t)n_events + 1), s);
    cudaMemsetAsync(d_track_offsets, 0, sizeof(int32_t), s);
  } else {
    int32_t *size = scratch + kOffSize, *keep = scratch + kOffKeep, *ksize = scratch + kOffKsize, *number = scratch + kOffNumber,
            *bsum = scratch + kOffBsum;
    const int g = (n_hits + 255) / 256;
    // the array still holds the previous call's values: the two accumulated arrays start from zero, the others are
    // written in full before they are read
    cudaMemsetAsync(size, 0, sizeof(int32_t) * (size_t)n_hits, s);
    cudaMemsetAsync(ksize, 0, sizeof(int32_t) * (size_t)n_hits, s);
    st_size_kernel<<<g, 256, 0, s>>>(d_track_id, n_hits, size);
    st_keep_kernel<<<g, 256, 0, s>>>(d_track_id, size, n_hits, min_hits, keep);
    exclusive_scan(keep, n_hits, number, d_n_tracks, bsum, s);
    st_index_kernel<<<g, 256, 0, s>>>(d_track_id, size, number, n_hits, min_hits, d_track_index, ksize);
    exclusive_scan(ksize, n_hits, d_track_offsets, nullptr, bsum, s);           // entries past n_tracks repeat the total
    st_event_kernel<<<(n_events + 256) / 256, 256, 0, s>>>(d_event_offsets, number, n_events, n_hits, d_event_track_offsets);
    st_fill_kernel<<<(n_events + 7) / 8, 256, 0, s>>>(d_track_index, d_track_offsets, d_event_offsets, d_event_track_offsets,
                                                      n_events, n_hits, keep, d_track_hits);   // keep is free again: cursors
  }
  const cudaError_t e = cudaGetLastError();
  if (e != cudaSuccess) return fail(ETX_ERR_CUDA, "launch failed", e);
  return ETX_OK;
}

extern "C" const char* etx_tracks_static_error(void) { return g_error; }
