// Track building from triplets, phases (3)-(4) (sec. 5.4: "Third, a new track is formed for each
// remaining articulation, effectively duplicating the shared set of connected edges.  Finally, edges are replaced by
// their corresponding hits"; Fig. 6; R30, R31), on the device, after etx_triplet_components:
//
//   input   edge_comp [E]      name of the set of connected edges a kept edge belongs to (-1: edge below threshold)
//           shared [ns][2]     the shared articulations as (set of first, set of second)
//   (3)     every shared articulation (X, Y) is a track candidate "set X united with set Y"; a set no shared
//           articulation touches is a candidate by itself
//   (4)     a candidate's hits are the end points of its edges
//   R31     hits ascend inside a track, candidates with fewer than min_hits hits are dropped, identical hit lists are
//           kept once, tracks are ordered lexicographically by hit list
//
// All integer work on sets, so the result does not depend on the order in which threads get there.  Written from the
// paper's prose and the two readings above; it shares nothing with oracle/ (which checks it).
//
// How.  A hit touches few sets (those of its in- and out-edges), so the hit lists of the sets are built per hit from
// the CSR / CSC of the hit graph: count the distinct sets per hit, prefix-sum per set, and let one warp per event place
// the event's hits in ascending order (sets never cross an event, R8).  A candidate is never materialised: its hit list
// is a two-way merge of the ascending lists of X and Y, walked wherever it is needed (length, first hit, comparison,
// final write).  Ordering: a list's first element is its smallest hit, so candidates are bucketed by first hit
// (count, prefix sum, fill) and every bucket -- a handful of candidates, those of tracks that start on the same hit --
// is sorted and de-duplicated by one thread; buckets in ascending hit order are then the lexicographic order.
#include "etx_internal.h"

namespace etx {
namespace {

constexpr int kTtThreads = 256;
constexpr int kTtItems = 8;
constexpr int kTtChunk = kTtThreads * kTtItems;

// ---- exclusive prefix sum over n elements (n known on the host), with a block-sum buffer of this stage's own ----------
__device__ __forceinline__ int tt_block_exclusive(int v, int* total) {
  __shared__ int wsum[kTtThreads / 32];
  const int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
  int incl = v;
#pragma unroll
  for (int o = 1; o < 32; o <<= 1) { const int y = __shfl_up_sync(0xffffffffu, incl, o); if (lane >= o) incl += y; }
  if (lane == 31) wsum[w] = incl;
  __syncthreads();
  int before = 0, all = 0;
#pragma unroll
  for (int i = 0; i < kTtThreads / 32; ++i) { const int s = wsum[i]; if (i < w) before += s; all += s; }
  __syncthreads();
  *total = all;
  return before + incl - v;
}
__global__ void __launch_bounds__(kTtThreads) tt_scan_sums_kernel(const int32_t* __restrict__ in, int n, int32_t* __restrict__ bsum) {
  const int first = blockIdx.x * kTtChunk + threadIdx.x * kTtItems;
  int v = 0;
#pragma unroll
  for (int j = 0; j < kTtItems; ++j) if (first + j < n) v += in[first + j];
  int tot;
  tt_block_exclusive(v, &tot);
  if (threadIdx.x == 0) bsum[blockIdx.x] = tot;
}
__global__ void __launch_bounds__(kTtThreads) tt_scan_bsum_kernel(int32_t* __restrict__ bsum, int nb) {   // one block
  int carry = 0;
  for (int b0 = 0; b0 < nb; b0 += kTtThreads) {
    const int i = b0 + threadIdx.x;
    int tot;
    const int ex = tt_block_exclusive(i < nb ? bsum[i] : 0, &tot);
    if (i < nb) bsum[i] = carry + ex;
    carry += tot;
  }
}
__global__ void __launch_bounds__(kTtThreads) tt_scan_write_kernel(const int32_t* __restrict__ in, int n, const int32_t* __restrict__ bsum,
                                                                   int32_t* __restrict__ out, int32_t* __restrict__ total) {
  const int first = blockIdx.x * kTtChunk + threadIdx.x * kTtItems;
  int x[kTtItems], v = 0;
#pragma unroll
  for (int j = 0; j < kTtItems; ++j) { x[j] = first + j < n ? in[first + j] : 0; v += x[j]; }
  int tot;
  int run = tt_block_exclusive(v, &tot) + bsum[blockIdx.x];
#pragma unroll
  for (int j = 0; j < kTtItems; ++j) {
    const int i = first + j;
    if (i < n) out[i] = run;
    run += x[j];
    if (i == n - 1) { out[n] = run; if (total) *total = run; }
  }
}
// out[0..n] = exclusive prefix sums of in[0..n), n >= 1; optionally *total = out[n]
void tt_scan(etx_ctx* c, const int32_t* in, int n, int32_t* out, int32_t* total, cudaStream_t s) {
  const int nb = (n + kTtChunk - 1) / kTtChunk;
  tt_scan_sums_kernel<<<nb, kTtThreads, 0, s>>>(in, n, c->tt_scan_tmp);
  tt_scan_bsum_kernel<<<1, kTtThreads, 0, s>>>(c->tt_scan_tmp, nb);
  tt_scan_write_kernel<<<nb, kTtThreads, 0, s>>>(in, n, c->tt_scan_tmp, out, total);
  c->launches += 3;
}

// ---- the sets a hit touches -------------------------------------------------------------------------------------------
// Incident edges of hit h: its out-edges (CSR row, edge ids row_ptr[h] ..) then its in-edges (CSC column, in_edge[]).
struct Incident {
  const int32_t* in_edge; const int32_t* comp;
  int row0, od, col0, deg;
  __device__ Incident(const int32_t* row_ptr, const int32_t* col_ptr, const int32_t* in_edge_, const int32_t* comp_, int h)
      : in_edge(in_edge_), comp(comp_) {
    row0 = row_ptr[h]; od = row_ptr[h + 1] - row0; col0 = col_ptr[h]; deg = od + col_ptr[h + 1] - col0;
  }
  __device__ int set_of(int t) const { return comp[t < od ? row0 + t : in_edge[col0 + t - od]]; }
  // the set of incident edge t if t is the first incident edge of that set (and the edge is kept), else -1
  __device__ int new_set(int t) const {
    const int x = set_of(t);
    if (x < 0) return -1;
    for (int u = 0; u < t; ++u) if (set_of(u) == x) return -1;
    return x;
  }
};

__global__ void tt_count_kernel(const int32_t* __restrict__ row_ptr, const int32_t* __restrict__ col_ptr,
                                const int32_t* __restrict__ in_edge, const int32_t* __restrict__ comp, int n_hits,
                                int32_t* __restrict__ set_size) {
  const int h = blockIdx.x * blockDim.x + threadIdx.x;
  if (h >= n_hits) return;
  const Incident inc(row_ptr, col_ptr, in_edge, comp, h);
  for (int t = 0; t < inc.deg; ++t) { const int x = inc.new_set(t); if (x >= 0) atomicAdd(&set_size[x], 1); }
}

// One warp per event walks the event's hits in ascending order, 32 per step; in every round each lane brings the next
// set its hit touches, lanes that bring the same set are ranked by lane (= by hit) and the lowest moves the set's
// cursor.  Inside a round the hits of a set ascend; two rounds of one step may interleave, so a list comes out sorted
// up to displacements of a few dozen places, which tt_sort_sets_kernel removes.  Only this warp touches the cursors of
// its event's sets.
__global__ void __launch_bounds__(256)
tt_fill_kernel(const int32_t* __restrict__ row_ptr, const int32_t* __restrict__ col_ptr, const int32_t* __restrict__ in_edge,
               const int32_t* __restrict__ comp, const int32_t* __restrict__ event_off, int n_events, int32_t* cursor,
               int32_t* __restrict__ set_hits) {
  const int e = blockIdx.x * 8 + (threadIdx.x >> 5), lane = threadIdx.x & 31;
  if (e >= n_events) return;
  const int h0 = event_off[e], h1 = event_off[e + 1];
  volatile int32_t* cur = cursor;
  for (int i0 = h0; i0 < h1; i0 += 32) {
    const int h = i0 + lane;
    const bool valid = h < h1;
    const Incident inc(row_ptr, col_ptr, in_edge, comp, valid ? h : h0);
    int t = 0;
    while (true) {
      int x = -1;
      if (valid) while (t < inc.deg && x < 0) x = inc.new_set(t++);
      const unsigned active = __ballot_sync(0xffffffffu, x >= 0);
      if (!active) break;
      if (x >= 0) {
        const unsigned peers = __match_any_sync(active, x);
        const int leader = __ffs(peers) - 1, rank = __popc(peers & ((1u << lane) - 1u));
        int pos = 0;
        if (lane == leader) { pos = cur[x]; cur[x] = pos + __popc(peers); }
        pos = __shfl_sync(peers, pos, leader);
        set_hits[pos + rank] = h;
      }
      __syncwarp();
    }
  }
}

__global__ void tt_sort_sets_kernel(const int32_t* __restrict__ set_off, int n_sets, int32_t* __restrict__ set_hits) {
  const int x = blockIdx.x * blockDim.x + threadIdx.x;
  if (x >= n_sets) return;
  const int a = set_off[x], b = set_off[x + 1];
  for (int i = a + 1; i < b; ++i) {                              // insertion sort of an almost sorted list
    const int v = set_hits[i];
    int j = i - 1;
    while (j >= a && set_hits[j] > v) { set_hits[j + 1] = set_hits[j]; --j; }
    set_hits[j + 1] = v;
  }
}

__global__ void tt_touch_kernel(const int32_t* __restrict__ shared, const int32_t* __restrict__ n_shared, int cap, int32_t* __restrict__ touched) {
  const int ns = max(0, min(*n_shared, cap));
  for (int i = blockIdx.x * blockDim.x + threadIdx.x; i < ns; i += gridDim.x * blockDim.x) {
    touched[shared[2 * (size_t)i]] = 1; touched[shared[2 * (size_t)i + 1]] = 1;
  }
}

// ---- candidates ---------------------------------------------------------------------------------------------------------
// Ascending, duplicate-free walk over the hits of set x united with set y (y < 0: x alone).
struct Walk {
  const int32_t *a, *b;
  int na, nb, i, j;
  __device__ Walk(const int32_t* set_off, const int32_t* set_hits, int x, int y) : i(0), j(0) {
    a = set_hits + set_off[x]; na = set_off[x + 1] - set_off[x];
    if (y >= 0 && y != x) { b = set_hits + set_off[y]; nb = set_off[y + 1] - set_off[y]; } else { b = a; nb = 0; }
  }
  __device__ int next() {                                        // -1 at the end
    if (i < na && (j >= nb || a[i] <= b[j])) { const int v = a[i++]; if (j < nb && b[j] == v) ++j; return v; }
    if (j < nb) return b[j++];
    return -1;
  }
};

// Candidate number q: q < ns is shared articulation q; q >= ns is the set q - ns by itself (valid if it has hits and no
// shared articulation touches it).  -> (x, y), false if q is no candidate.
__device__ __forceinline__ bool tt_candidate(long long q, int ns, int n_sets, const int32_t* shared, const int32_t* set_off,
                                             const int32_t* touched, int* x, int* y) {
  if (q < ns) { *x = shared[2 * q]; *y = shared[2 * q + 1]; return *x >= 0 && *y >= 0; }
  const long long s = q - ns;
  if (s >= n_sets) return false;
  *x = (int)s; *y = -1;
  return set_off[s + 1] > set_off[s] && !touched[s];
}

// FILL = false: count the candidates with >= min_hits hits per first hit; FILL = true: place their numbers
template <bool FILL>
__global__ void tt_bucket_kernel(const int32_t* __restrict__ shared, const int32_t* __restrict__ n_shared, int cap, int n_sets,
                                 const int32_t* __restrict__ set_off, const int32_t* __restrict__ set_hits,
                                 const int32_t* __restrict__ touched, int min_hits, int32_t* bucket_cnt,
                                 const int32_t* __restrict__ bucket_off, int32_t* __restrict__ bucket_cand) {
  const int ns = max(0, min(*n_shared, cap));
  const long long n_q = (long long)ns + n_sets, stride = (long long)gridDim.x * blockDim.x;
  for (long long q = (long long)blockIdx.x * blockDim.x + threadIdx.x; q < n_q; q += stride) {
    int x, y;
    if (!tt_candidate(q, ns, n_sets, shared, set_off, touched, &x, &y)) continue;
    Walk w(set_off, set_hits, x, y);
    const int first = w.next();
    if (first < 0) continue;
    int len = 1;
    while (len < min_hits && w.next() >= 0) ++len;
    if (len < min_hits) continue;
    const int p = atomicAdd(&bucket_cnt[first], 1);
    if (FILL) bucket_cand[bucket_off[first] + p] = (int)q;
  }
}

// One thread per first hit: order the bucket's candidates lexicographically by hit list, keep one of every run of equal
// lists (compacted to the front of the bucket), report how many are left.
__global__ void tt_bucket_sort_kernel(const int32_t* __restrict__ shared, const int32_t* __restrict__ n_shared, int cap, int n_sets,
                                      const int32_t* __restrict__ set_off, const int32_t* __restrict__ set_hits,
                                      const int32_t* __restrict__ bucket_off, int n_hits, int32_t* __restrict__ bucket_cand,
                                      int32_t* __restrict__ kept) {
  const int h = blockIdx.x * blockDim.x + threadIdx.x;
  if (h >= n_hits) return;
  const int ns = max(0, min(*n_shared, cap));
  const int a = bucket_off[h], b = bucket_off[h + 1];
  if (a == b) { kept[h] = 0; return; }
  auto cmp = [&](int q1, int q2) {                               // <0, 0, >0; a proper prefix sorts first
    int x1, y1, x2, y2;
    if (q1 < ns) { x1 = shared[2 * (size_t)q1]; y1 = shared[2 * (size_t)q1 + 1]; } else { x1 = q1 - ns; y1 = -1; }
    if (q2 < ns) { x2 = shared[2 * (size_t)q2]; y2 = shared[2 * (size_t)q2 + 1]; } else { x2 = q2 - ns; y2 = -1; }
    Walk w1(set_off, set_hits, x1, y1), w2(set_off, set_hits, x2, y2);
    while (true) {
      const int u = w1.next(), v = w2.next();
      if (u != v) return u < 0 ? -1 : v < 0 ? 1 : (u < v ? -1 : 1);
      if (u < 0) return 0;
    }
  };
  for (int i = a + 1; i < b; ++i) {
    const int v = bucket_cand[i];
    int j = i - 1;
    while (j >= a && cmp(bucket_cand[j], v) > 0) { bucket_cand[j + 1] = bucket_cand[j]; --j; }
    bucket_cand[j + 1] = v;
  }
  int n = 1;
  for (int i = a + 1; i < b; ++i)
    if (cmp(bucket_cand[a + n - 1], bucket_cand[i]) != 0) bucket_cand[a + n++] = bucket_cand[i];
  kept[h] = n;
}

// WRITE = false: the length of every track, in its final position; WRITE = true: its hits
template <bool WRITE>
__global__ void tt_emit_kernel(const int32_t* __restrict__ shared, const int32_t* __restrict__ n_shared, int cap,
                               const int32_t* __restrict__ set_off, const int32_t* __restrict__ set_hits,
                               const int32_t* __restrict__ bucket_off, const int32_t* __restrict__ bucket_cand,
                               const int32_t* __restrict__ kept, const int32_t* __restrict__ track_no, int n_hits,
                               int track_cap, int hit_cap, int32_t* __restrict__ track_len, const int32_t* __restrict__ track_off,
                               int32_t* __restrict__ track_hits) {
  const int h = blockIdx.x * blockDim.x + threadIdx.x;
  if (h >= n_hits) return;
  const int ns = max(0, min(*n_shared, cap));
  for (int j = 0; j < kept[h]; ++j) {
    const int t = track_no[h] + j;
    if (t >= track_cap) return;
    const int q = bucket_cand[bucket_off[h] + j];
    int x, y;
    if (q < ns) { x = shared[2 * (size_t)q]; y = shared[2 * (size_t)q + 1]; } else { x = q - ns; y = -1; }
    Walk w(set_off, set_hits, x, y);
    if (!WRITE) {
      int len = 0;
      while (w.next() >= 0) ++len;
      track_len[t] = len;
    } else {
      int pos = track_off[t];
      for (int v = w.next(); v >= 0 && pos < hit_cap; v = w.next()) track_hits[pos++] = v;
    }
  }
}

__global__ void tt_counts_kernel(const int32_t* __restrict__ track_no, int n_hits, const int32_t* __restrict__ track_off, int track_cap,
                                 int hit_cap, int32_t* __restrict__ counts) {
  const int n_tracks = track_no[n_hits], total = track_off[track_cap];
  counts[0] = n_tracks; counts[1] = total; counts[2] = (n_tracks > track_cap || total > hit_cap) ? 1 : 0;
}

}  // namespace

void launch_triplet_tracks(etx_ctx* c, int n_events, int n_hits, int min_hits, cudaStream_t s) {
  const int n_sets = c->max_edges, cap = c->hp.max_triplets, track_cap = c->tt_track_cap, hit_cap = c->tt_hit_cap;
  const size_t st = (size_t)c->hp.max_hits + 1;
  // scratch shared with the calls that ran before: the union-find and counting arrays of etx_triplet_components and the
  // per-hit count / offset arrays of etx_triplets are free once those calls' kernels are done (same stream)
  int32_t *set_size = c->tc_succ, *touched = c->tc_par2, *cursor = c->tc_par1;
  int32_t *bucket_cnt = c->trip_cnt, *kept = c->trip_cnt + st, *track_len = c->tt_track_len;
  int32_t *bucket_off = c->trip_off, *track_no = c->trip_off + st;
  if (n_hits == 0 || n_events == 0) {
    cudaMemsetAsync(c->tt_counts, 0, 4 * sizeof(int32_t), s);
    cudaMemsetAsync(c->tt_track_off, 0, sizeof(int32_t), s);
    return;
  }
  cudaMemsetAsync(set_size, 0, sizeof(int32_t) * (size_t)n_sets, s);
  cudaMemsetAsync(touched, 0, sizeof(int32_t) * (size_t)n_sets, s);
  cudaMemsetAsync(bucket_cnt, 0, sizeof(int32_t) * (size_t)n_hits, s);
  cudaMemsetAsync(track_len, 0, sizeof(int32_t) * (size_t)track_cap, s);
  const int gh = (n_hits + 127) / 128, g = c->sm_count * 8;
  // (4) first: the hit list of every set of connected edges
  tt_count_kernel<<<gh, 128, 0, s>>>(c->row_ptr, c->col_ptr, c->in_edge, c->tc_comp, n_hits, set_size);
  tt_scan(c, set_size, n_sets, c->tt_set_off, nullptr, s);
  cudaMemcpyAsync(cursor, c->tt_set_off, sizeof(int32_t) * (size_t)n_sets, cudaMemcpyDeviceToDevice, s);
  tt_fill_kernel<<<(n_events + 7) / 8, 256, 0, s>>>(c->row_ptr, c->col_ptr, c->in_edge, c->tc_comp, c->event_off, n_events, cursor, c->tt_set_hits);
  tt_sort_sets_kernel<<<(n_sets + 127) / 128, 128, 0, s>>>(c->tt_set_off, n_sets, c->tt_set_hits);
  // (3) candidates, bucketed by their first hit
  tt_touch_kernel<<<g, 256, 0, s>>>(c->tc_shared, c->tc_n_shared, cap, touched);
  tt_bucket_kernel<false><<<g, 256, 0, s>>>(c->tc_shared, c->tc_n_shared, cap, n_sets, c->tt_set_off, c->tt_set_hits, touched, min_hits,
                                            bucket_cnt, nullptr, nullptr);
  tt_scan(c, bucket_cnt, n_hits, bucket_off, nullptr, s);
  cudaMemsetAsync(bucket_cnt, 0, sizeof(int32_t) * (size_t)n_hits, s);
  tt_bucket_kernel<true><<<g, 256, 0, s>>>(c->tc_shared, c->tc_n_shared, cap, n_sets, c->tt_set_off, c->tt_set_hits, touched, min_hits,
                                           bucket_cnt, bucket_off, c->tt_bucket_cand);
  // R31: order, duplicates, final numbering, lengths, hits
  tt_bucket_sort_kernel<<<gh, 128, 0, s>>>(c->tc_shared, c->tc_n_shared, cap, n_sets, c->tt_set_off, c->tt_set_hits, bucket_off, n_hits,
                                           c->tt_bucket_cand, kept);
  tt_scan(c, kept, n_hits, track_no, nullptr, s);
  tt_emit_kernel<false><<<gh, 128, 0, s>>>(c->tc_shared, c->tc_n_shared, cap, c->tt_set_off, c->tt_set_hits, bucket_off, c->tt_bucket_cand, kept,
                                           track_no, n_hits, track_cap, hit_cap, track_len, nullptr, nullptr);
  tt_scan(c, track_len, track_cap, c->tt_track_off, nullptr, s);
  tt_emit_kernel<true><<<gh, 128, 0, s>>>(c->tc_shared, c->tc_n_shared, cap, c->tt_set_off, c->tt_set_hits, bucket_off, c->tt_bucket_cand, kept,
                                          track_no, n_hits, track_cap, hit_cap, nullptr, c->tt_track_off, c->tt_track_hits);
  tt_counts_kernel<<<1, 1, 0, s>>>(track_no, n_hits, c->tt_track_off, track_cap, hit_cap, c->tt_counts);
  c->launches += 10;
}

}  // namespace etx
