// Graph stages of the ETX4VELO hot path on sm_100a: S0 plane offsets, S2 plane-restricted k-NN,
// S3 edge compaction + CSC, S5 threshold + connected components.  All integer / index work here is
// bit-exact by construction; the only floating point is Eq.(1) in a pinned operation order.
#include "etx_internal.h"

namespace etx {

// --------------------------------------------------------------------------------------------------------
// C1 (PAPER.md L107 fn.5; R1): f = ((x,y,z) + offset) / div, one IEEE add and one correctly
// rounded division.  Stored once as float4 so every later stage gathers 16 B per hit.
struct FeatArgs { float o[3], d[3], co[3], cd[3]; };

// phi = atan2(y, x) in fp32 as DESIGN.md R27 states it (every step one correctly rounded operation, in this order):
// a = min(|x|,|y|) / max(|x|,|y|), an odd polynomial in a on [0,1] (Horner in a*a with fma, degree 8), then the
// octant, half-plane and sign corrections.  |phi - atan2| <= 5e-7.
__device__ __forceinline__ float atan2_r27(float y, float x) {
  const float ax = fabsf(x), ay = fabsf(y);
  const float mx = ax > ay ? ax : ay, mn = ax > ay ? ay : ax;
  const float a = mx > 0.0f ? __fdiv_rn(mn, mx) : 0.0f;
  const float s = __fmul_rn(a, a);
  float q = 0x1.6a9512p-9f;
  q = __fmaf_rn(q, s, -0x1.01bda4p-6f);
  q = __fmaf_rn(q, s, 0x1.593100p-5f);
  q = __fmaf_rn(q, s, -0x1.316ecap-4f);
  q = __fmaf_rn(q, s, 0x1.b2edb0p-4f);
  q = __fmaf_rn(q, s, -0x1.22c55ap-3f);
  q = __fmaf_rn(q, s, 0x1.996efcp-3f);
  q = __fmaf_rn(q, s, -0x1.55548ep-2f);
  q = __fmaf_rn(q, s, 1.0f);
  float p = __fmul_rn(a, q);
  if (ay > ax) p = __fsub_rn(1.57079637f, p);
  if (x < 0.0f) p = __fsub_rn(3.14159274f, p);
  return copysignf(p, y);
}

template <bool CYL>
__global__ void features_kernel(const float* __restrict__ xyz, float4* __restrict__ feat, float4* __restrict__ feat_emb,
                                int32_t* __restrict__ deg, int n, FeatArgs a) {
  int i = blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= n) return;
  deg[i] = 0;        // S2 writes the out-degree of every hit of every (event, plane) bucket; a hit of a rejected batch
                     // (planes out of order / out of range) may belong to none and must not keep a stale value
  float x = xyz[3 * (size_t)i], y = xyz[3 * (size_t)i + 1], z = xyz[3 * (size_t)i + 2];
  feat[i] = make_float4(__fdiv_rn(__fadd_rn(x, a.o[0]), a.d[0]), __fdiv_rn(__fadd_rn(y, a.o[1]), a.d[1]),
                        __fdiv_rn(__fadd_rn(z, a.o[2]), a.d[2]), 0.0f);
  if (CYL) {                                              // L96: the embedding reads normalised (r, phi, z)
    const float r = __fsqrt_rn(__fmaf_rn(y, y, __fmul_rn(x, x)));
    const float phi = atan2_r27(y, x);
    feat_emb[i] = make_float4(__fdiv_rn(__fadd_rn(r, a.co[0]), a.cd[0]), __fdiv_rn(__fadd_rn(phi, a.co[1]), a.cd[1]),
                              __fdiv_rn(__fadd_rn(z, a.co[2]), a.cd[2]), 0.0f);
  }
}

void launch_features(etx_ctx* c, const float* xyz, int n_hits, cudaStream_t s) {
  if (n_hits == 0) return;
  const etx_hyperparams& hp = c->hp;
  FeatArgs a;
  for (int i = 0; i < 3; ++i) {
    a.o[i] = hp.norm_offset[i]; a.d[i] = hp.norm_div[i]; a.co[i] = hp.cyl_offset[i]; a.cd[i] = hp.cyl_div[i];
  }
  if (hp.emb_input) features_kernel<true><<<(n_hits + 255) / 256, 256, 0, s>>>(xyz, c->feat, c->feat_emb, c->deg, n_hits, a);
  else features_kernel<false><<<(n_hits + 255) / 256, 256, 0, s>>>(xyz, c->feat, c->feat_emb, c->deg, n_hits, a);
  c->launches++;
}

// --------------------------------------------------------------------------------------------------------
// S0 (L26, L223, L257): plane_off[e][p] = first hit of event e with plane >= p (lower bound in the sorted
// plane array); entry P is the event's end.  One thread per (event, p).
__global__ void plane_offsets_kernel(const int32_t* __restrict__ plane, const int32_t* __restrict__ event_off,
                                     int n_events, int P, int32_t* __restrict__ plane_off) {
  int i = blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= n_events * (P + 1)) return;
  int e = i / (P + 1), p = i % (P + 1);
  int lo = event_off[e], hi = event_off[e + 1];
  while (lo < hi) {
    int mid = (lo + hi) >> 1;
    if (plane[mid] < p) lo = mid + 1; else hi = mid;
  }
  plane_off[i] = lo;
}

void launch_plane_offsets(etx_ctx* c, const int32_t* plane, int n_events, cudaStream_t s) {
  int n = n_events * (c->hp.n_planes + 1);
  if (n == 0) return;
  plane_offsets_kernel<<<(n + 255) / 256, 256, 0, s>>>(plane, c->event_off, n_events, c->hp.n_planes, c->plane_off);
  c->launches++;
}

// Input contract check (include/etx.h): plane in range, and non-decreasing except across an event boundary.
__global__ void validate_kernel(const int32_t* __restrict__ plane, const int32_t* __restrict__ event_off,
                                int n_events, int n_hits, int P, int32_t* __restrict__ flags) {
  int i = blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= n_hits) return;
  int p = plane[i];
  bool bad = p < 0 || p >= P;
  if (!bad && i + 1 < n_hits && plane[i + 1] < p) {
    int lo = 0, hi = n_events + 1;               // is i + 1 the start of some event?
    while (lo < hi) { int mid = (lo + hi) >> 1; if (event_off[mid] < i + 1) lo = mid + 1; else hi = mid; }
    bad = !(lo <= n_events && event_off[lo] == i + 1);
  }
  if (bad) atomicOr(&flags[0], 1);
}

void launch_validate(etx_ctx* c, const int32_t* plane, int n_events, int n_hits, cudaStream_t s) {
  if (n_hits == 0) return;
  validate_kernel<<<(n_hits + 255) / 256, 256, 0, s>>>(plane, c->event_off, n_events, n_hits, c->hp.n_planes, c->flags);
  c->launches++;
}

// --------------------------------------------------------------------------------------------------------
// S2 (L98 Eq.(1), L101, L257 sec. 7.2; R4-R8).  For hit q on plane p the candidates are the hits of the same
// event on planes p+1 .. min(p+w, P-1): one contiguous index range given by the plane offsets.  The result
// is the first min(k, #kept) candidates in ascending (d2, index) order, d2 < d2_max strict.
//
// The paper's kernel is one thread per query scanning global memory.  Here a CTA owns one (event, plane)
// bucket and stages the candidate range through shared memory in tiles (so capacity never depends on the
// window size); one thread per query walks the tile in ascending candidate index, all lanes of a warp reading
// the same candidate (a shared-memory broadcast).  Each thread keeps its k best (d2, index) pairs sorted in
// registers.  Because the walk is in ascending index and the insertion is stable (a candidate goes behind
// every stored entry with d2 <= its own), the list is ordered by (d2, index) without ever comparing indices,
// and `d2 < worst` (strict) rejects exactly the candidates that lose under that order (R5).  The empty slots
// hold d2_max, so the radius cut `d2 < d2_max` (R6) is the same comparison.
template <int KCAP>
struct TopK {
  float key[KCAP];
  int idx[KCAP];
  __device__ __forceinline__ void init(float d2_max) {
#pragma unroll
    for (int s = 0; s < KCAP; ++s) { key[s] = d2_max; idx[s] = -1; }
  }
  // stable insertion into the ascending list of all KCAP slots; the entry pushed out of the last slot is dropped.
  // The first k entries of a top-KCAP list are the top-k list, so k < KCAP needs no special case (and no
  // run-time slot index, which would push the arrays into local memory).
  __device__ __forceinline__ void insert(float d2, int id) {
    // the list is ascending, so lt[s] = (d2 < key[s]) is monotone in s: slot s takes the new entry if it is the
    // first slot with lt, the old slot s-1 if lt[s-1] already held, and keeps its own otherwise.  Entries equal
    // to d2 stay in front of it (stable).  Walking down keeps key[s-1] / idx[s-1] old when slot s is written.
#pragma unroll
    for (int s = KCAP - 1; s > 0; --s) {
      const bool lt = d2 < key[s], ltp = d2 < key[s - 1];
      key[s] = lt ? (ltp ? key[s - 1] : d2) : key[s];
      idx[s] = lt ? (ltp ? idx[s - 1] : id) : idx[s];
    }
    const bool lt0 = d2 < key[0];
    key[0] = lt0 ? d2 : key[0];
    idx[0] = lt0 ? id : idx[0];
  }
  __device__ __forceinline__ float worst() const { return key[KCAP - 1]; }
};

constexpr int kKnnThreads = 128;
constexpr int kKnnTile = 1024;       // candidates per shared-memory tile (16 KB)

// Eq.(1) in the pinned order: t0*t0, then fma(t_i, t_i, d2)   (R4)
__device__ __forceinline__ float knn_d2(const float4 a, const float4 b) {
  float t = __fsub_rn(a.x, b.x);
  float d2 = __fmul_rn(t, t);
  t = __fsub_rn(a.y, b.y); d2 = __fmaf_rn(t, t, d2);
  t = __fsub_rn(a.z, b.z); d2 = __fmaf_rn(t, t, d2);
  t = __fsub_rn(a.w, b.w); d2 = __fmaf_rn(t, t, d2);
  return d2;
}

template <int KCAP>
__global__ void __launch_bounds__(kKnnThreads)
knn_kernel(const float4* __restrict__ emb, const int32_t* __restrict__ plane_off, int P, int k, int w,
           float d2_max, int32_t* __restrict__ nbr, int32_t* __restrict__ deg, const int32_t* __restrict__ only) {
  __shared__ float4 cand[kKnnTile];
  const int bucket = blockIdx.x;                 // e * P + p
  if (only && !only[bucket]) return;             // second pass after knn_cut_kernel: flagged buckets only
  const int e = bucket / P, p = bucket % P;
  const int32_t* po = plane_off + (size_t)e * (P + 1);
  const int q_lo = po[p], q_hi = po[p + 1];
  if (q_lo == q_hi) return;
  const int p_hi = min(p + w, P - 1);
  const int c_lo = po[p + 1], c_hi = (p + 1 <= p_hi) ? po[p_hi + 1] : po[p + 1];
  const bool single = (c_hi - c_lo) <= kKnnTile;   // the usual case: stage the window once for every pass
  if (single) {
    for (int i = threadIdx.x; i < c_hi - c_lo; i += kKnnThreads) cand[i] = emb[c_lo + i];
    __syncthreads();
  }
  for (int q0 = q_lo; q0 < q_hi; q0 += kKnnThreads) {
    const int q = q0 + threadIdx.x;
    const bool active = q < q_hi && (!only || deg[q] < 0);    // second pass: only the hits knn_cut_kernel gave up on
    const float4 a = active ? emb[q] : make_float4(0.f, 0.f, 0.f, 0.f);
    TopK<KCAP> top;
    top.init(d2_max);
    float worst = d2_max;
    for (int t0 = c_lo; t0 < c_hi; t0 += kKnnTile) {
      const int nt = min(kKnnTile, c_hi - t0);
      if (!single) {
        __syncthreads();
        for (int i = threadIdx.x; i < nt; i += kKnnThreads) cand[i] = emb[t0 + i];
        __syncthreads();
      }
      if (active) {
        int i = 0;
        for (; i + 4 <= nt; i += 4) {
          const float d0 = knn_d2(a, cand[i]), d1 = knn_d2(a, cand[i + 1]);
          const float d2 = knn_d2(a, cand[i + 2]), d3 = knn_d2(a, cand[i + 3]);
          if (d0 < worst) { top.insert(d0, t0 + i); worst = top.worst(); }
          if (d1 < worst) { top.insert(d1, t0 + i + 1); worst = top.worst(); }
          if (d2 < worst) { top.insert(d2, t0 + i + 2); worst = top.worst(); }
          if (d3 < worst) { top.insert(d3, t0 + i + 3); worst = top.worst(); }
        }
        for (; i < nt; ++i) {
          const float d0 = knn_d2(a, cand[i]);
          if (d0 < worst) { top.insert(d0, t0 + i); worst = top.worst(); }
        }
      }
    }
    if (active) {
      int cnt = 0;
#pragma unroll
      for (int s = 0; s < KCAP; ++s) {
        if (s < k) {
          if (top.idx[s] >= 0) { nbr[(size_t)q * k + s] = top.idx[s]; ++cnt; }   // slots past deg[q] are never read
        }
      }
      deg[q] = cnt;
    }
  }
}

// With a finite radius cut (the paper's regime, L101 / L257: ~14 of a hit's ~160 candidates lie inside d2_max and
// "less than 0.1 % of hits have more than 50 neighbours") the sorted insertion is the wrong tool: almost every
// candidate is rejected by the cut, yet the insertion code runs whenever any lane of the warp accepts one.  This
// kernel only collects the candidates inside the cut, in scan order, in a per-thread shared-memory list of kKnnBuf
// entries, then sorts that short list by d2 (stable, so equal distances stay in ascending index order: R5) and
// writes its first k entries.  A hit with more than kKnnBuf candidates inside the cut gets deg = -1 and its bucket
// a flag in `redo`; knn_kernel, which is exact for any count, then does those hits.
constexpr int kKnnBuf = 64;            // >= the largest k
constexpr int kKnnCutTile = 512;       // candidates per shared-memory tile (8 KB)
constexpr int kKnnCutThreads = 96;     // a VELO bucket holds ~80 hits: three full warps; 56 KB per block, four blocks per SM

__global__ void __launch_bounds__(kKnnCutThreads)
knn_cut_kernel(const float4* __restrict__ emb, const int32_t* __restrict__ plane_off, int P, int k, int w,
               float d2_max, int32_t* __restrict__ nbr, int32_t* __restrict__ deg, int32_t* __restrict__ redo) {
  extern __shared__ float4 knn_smem[];
  float4* cand = knn_smem;                                              // [kKnnCutTile]
  float* bkey = reinterpret_cast<float*>(knn_smem + kKnnCutTile);       // [kKnnBuf][kKnnCutThreads]
  int* bidx = reinterpret_cast<int*>(bkey + kKnnBuf * kKnnCutThreads);     // [kKnnBuf][kKnnCutThreads]
  const int bucket = blockIdx.x, tid = threadIdx.x;
  const int e = bucket / P, p = bucket % P;
  const int32_t* po = plane_off + (size_t)e * (P + 1);
  const int q_lo = po[p], q_hi = po[p + 1];
  if (q_lo == q_hi) { if (tid == 0) redo[bucket] = 0; return; }
  const int p_hi = min(p + w, P - 1);
  const int c_lo = po[p + 1], c_hi = (p + 1 <= p_hi) ? po[p_hi + 1] : po[p + 1];
  const bool single = (c_hi - c_lo) <= kKnnCutTile;
  if (single) {
    for (int i = tid; i < c_hi - c_lo; i += kKnnCutThreads) cand[i] = emb[c_lo + i];
    __syncthreads();
  }
  int overflow = 0;
  for (int q0 = q_lo; q0 < q_hi; q0 += kKnnCutThreads) {
    const int q = q0 + tid;
    const bool active = q < q_hi;
    const float4 a = active ? emb[q] : make_float4(0.f, 0.f, 0.f, 0.f);
    int cnt = 0;
    for (int t0 = c_lo; t0 < c_hi; t0 += kKnnCutTile) {
      const int nt = min(kKnnCutTile, c_hi - t0);
      if (!single) {
        __syncthreads();
        for (int i = tid; i < nt; i += kKnnCutThreads) cand[i] = emb[t0 + i];
        __syncthreads();
      }
      if (active) {
#pragma unroll 4
        for (int i = 0; i < nt; ++i) {
          const float d = knn_d2(a, cand[i]);
          if (d < d2_max) {                                             // R6: strict
            if (cnt < kKnnBuf) { bkey[cnt * kKnnCutThreads + tid] = d; bidx[cnt * kKnnCutThreads + tid] = t0 + i; }
            ++cnt;
          }
        }
      }
    }
    // The lists of a warp's 32 hits are ordered one after the other by the whole warp: lane l ranks entries l and
    // l + 32 of the list (rank = entries with a smaller d2, or an equal d2 met earlier in the scan: R5) and writes the
    // entry to slot `rank` if that is one of the first k.  Ranking only reads the list, and the warp's cost is the sum
    // of the list lengths, not 32 times the longest one.
    const bool over = active && cnt > kKnnBuf;
    if (over) { overflow = 1; deg[q] = -1; }                            // knn_kernel redoes this hit
    const int my_n = (active && !over) ? cnt : 0;
    if (active && !over) deg[q] = min(cnt, k);                          // slots past deg[q] are never read
    __syncwarp();
    const int lane = tid & 31, wbase = tid & ~31;
    for (int l = 0; l < 32; ++l) {
      const int n = __shfl_sync(0xffffffffu, my_n, l);
      if (n == 0) continue;
      const int col = wbase + l;
      int32_t* out = nbr + (size_t)(q0 + col) * k;
      for (int i = lane; i < n; i += 32) {
        const float kd = bkey[i * kKnnCutThreads + col];
        int rank = 0;
        for (int j = 0; j < n; ++j) {
          const float kj = bkey[j * kKnnCutThreads + col];
          rank += (kj < kd) || (kj == kd && j < i);
        }
        if (rank < k) out[rank] = bidx[i * kKnnCutThreads + col];
      }
    }
    __syncwarp();                                                       // the lists are rewritten by the next batch
  }
  overflow = __syncthreads_or(overflow);
  if (tid == 0) redo[bucket] = overflow;
}

template <int KCAP>
static void knn_dispatch(etx_ctx* c, int n_buckets, const int32_t* only, cudaStream_t s) {
  const etx_hyperparams& hp = c->hp;
  knn_kernel<KCAP><<<n_buckets, kKnnThreads, 0, s>>>(c->emb, c->plane_off, hp.n_planes, hp.k, hp.window,
                                                    hp.d2_max, c->nbr, c->deg, only);
  c->launches++;
}

void launch_knn(etx_ctx* c, const int32_t* plane, int n_events, int n_hits, cudaStream_t s) {
  (void)plane;
  if (n_hits == 0 || n_events == 0) return;
  const etx_hyperparams& hp = c->hp;
  const int nb = n_events * hp.n_planes;
  const int k = hp.k;
  const int32_t* only = nullptr;
  if (isfinite(hp.d2_max)) {
    constexpr int smem = kKnnCutTile * (int)sizeof(float4) + kKnnBuf * kKnnCutThreads * 8;
    opt_in_smem(c, knn_cut_kernel, smem);
    knn_cut_kernel<<<nb, kKnnCutThreads, smem, s>>>(c->emb, c->plane_off, hp.n_planes, k, hp.window, hp.d2_max, c->nbr, c->deg, c->knn_redo);
    c->launches++;
    only = c->knn_redo;
  }
  if (k <= 4) knn_dispatch<4>(c, nb, only, s);
  else if (k <= 10) knn_dispatch<10>(c, nb, only, s);
  else if (k <= 16) knn_dispatch<16>(c, nb, only, s);
  else if (k <= 32) knn_dispatch<32>(c, nb, only, s);
  else knn_dispatch<64>(c, nb, only, s);
}

// --------------------------------------------------------------------------------------------------------
// S3 (L74-76, L137; R9): exclusive scan of the out-degrees -> row_ptr, E; pack (src, dst) in (src asc, rank asc)
// order; in-degree histogram -> col_ptr; in_edge = edge ids grouped by dst, ascending inside a group.
constexpr int kScanThreads = 256;
constexpr int kScanItems = 8;                       // per thread
constexpr int kScanChunk = kScanThreads * kScanItems;

__device__ __forceinline__ int block_exclusive_scan(int v, int* total) {   // blockDim = kScanThreads
  __shared__ int warp_sums[kScanThreads / 32];
  const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
  int x = v;
#pragma unroll
  for (int o = 1; o < 32; o <<= 1) { int y = __shfl_up_sync(0xffffffffu, x, o); if (lane >= o) x += y; }
  if (lane == 31) warp_sums[wid] = x;
  __syncthreads();
  if (wid == 0) {
    int s = lane < kScanThreads / 32 ? warp_sums[lane] : 0;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) { int y = __shfl_up_sync(0xffffffffu, s, o); if (lane >= o) s += y; }
    if (lane < kScanThreads / 32) warp_sums[lane] = s;
  }
  __syncthreads();
  const int base = wid ? warp_sums[wid - 1] : 0;
  *total = warp_sums[kScanThreads / 32 - 1];
  __syncthreads();
  return base + x - v;
}

__global__ void __launch_bounds__(kScanThreads) scan_reduce_kernel(const int32_t* __restrict__ in, int n,
                                                                  int32_t* __restrict__ bsum) {
  const int base = blockIdx.x * kScanChunk;
  int v = 0;
#pragma unroll
  for (int j = 0; j < kScanItems; ++j) { int i = base + threadIdx.x * kScanItems + j; if (i < n) v += in[i]; }
  int tot; block_exclusive_scan(v, &tot);
  if (threadIdx.x == 0) bsum[blockIdx.x] = tot;
}

__global__ void __launch_bounds__(kScanThreads) scan_bsum_kernel(int32_t* __restrict__ bsum, int nb) {
  int carry = 0;                                   // single block, sequential over chunks of 256
  for (int b0 = 0; b0 < nb; b0 += kScanThreads) {
    int i = b0 + threadIdx.x;
    int v = i < nb ? bsum[i] : 0, tot;
    int ex = block_exclusive_scan(v, &tot);
    if (i < nb) bsum[i] = carry + ex;
    carry += tot;
  }
}

__global__ void __launch_bounds__(kScanThreads) scan_write_kernel(const int32_t* __restrict__ in, int n,
                                                                 const int32_t* __restrict__ bsum,
                                                                 int32_t* __restrict__ out, int32_t* __restrict__ total,
                                                                 const int32_t* __restrict__ reject) {
  const int base = blockIdx.x * kScanChunk;
  // validate_input found the batch out of contract: every prefix sum is 0, so E = 0 and no E-sized kernel runs
  const bool rejected = reject != nullptr && reject[0] != 0;
  int vals[kScanItems], v = 0;
#pragma unroll
  for (int j = 0; j < kScanItems; ++j) {
    int i = base + threadIdx.x * kScanItems + j;
    vals[j] = i < n ? in[i] : 0;
    v += vals[j];
  }
  int tot;
  int ex = block_exclusive_scan(v, &tot) + bsum[blockIdx.x];
#pragma unroll
  for (int j = 0; j < kScanItems; ++j) {
    int i = base + threadIdx.x * kScanItems + j;
    if (i < n) out[i] = rejected ? 0 : ex;
    ex += vals[j];
    if (i == n - 1) { out[n] = rejected ? 0 : ex; if (total) *total = rejected ? 0 : ex; }
  }
}

__global__ void scan_empty_kernel(int32_t* out, int32_t* total) { out[0] = 0; if (total) *total = 0; }

// out[0..n] = exclusive prefix sums of in[0..n); *total = out[n]
static void exclusive_scan(etx_ctx* c, const int32_t* in, int n, int32_t* out, int32_t* total, cudaStream_t s,
                           const int32_t* reject = nullptr) {
  if (n == 0) { scan_empty_kernel<<<1, 1, 0, s>>>(out, total); c->launches++; return; }
  const int nb = (n + kScanChunk - 1) / kScanChunk;
  scan_reduce_kernel<<<nb, kScanThreads, 0, s>>>(in, n, c->scan_tmp);
  scan_bsum_kernel<<<1, kScanThreads, 0, s>>>(c->scan_tmp, nb);
  scan_write_kernel<<<nb, kScanThreads, 0, s>>>(in, n, c->scan_tmp, out, total, reject);
  c->launches += 3;
}

__global__ void pack_edges_kernel(const int32_t* __restrict__ nbr, const int32_t* __restrict__ deg,
                                  const int32_t* __restrict__ row_ptr, int n_hits, int k,
                                  int32_t* __restrict__ src, int32_t* __restrict__ dst, const int32_t* __restrict__ reject) {
  size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= (size_t)n_hits * k || reject[0] != 0) return;
  int q = (int)(i / k), sidx = (int)(i % k);
  if (sidx < deg[q]) {
    int pos = row_ptr[q] + sidx;
    src[pos] = q;
    dst[pos] = nbr[i];
  }
}

// Large k with a radius cut leaves most of the k slots of a hit empty (cfg 5: ~15 of 50): sixteen lanes per hit walk
// its deg[q] filled slots instead of one thread per slot.
__global__ void pack_edges_sparse_kernel(const int32_t* __restrict__ nbr, const int32_t* __restrict__ deg,
                                         const int32_t* __restrict__ row_ptr, int n_hits, int k,
                                         int32_t* __restrict__ src, int32_t* __restrict__ dst, const int32_t* __restrict__ reject) {
  const size_t t = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
  const int q = (int)(t >> 4), l = (int)(t & 15);
  if (q >= n_hits || reject[0] != 0) return;
  const int n = deg[q], base = row_ptr[q];
  for (int sidx = l; sidx < n; sidx += 16) {
    src[base + sidx] = q;
    dst[base + sidx] = nbr[(size_t)q * k + sidx];
  }
}

void launch_pack_edges(etx_ctx* c, int n_hits, cudaStream_t s) {
  exclusive_scan(c, c->deg, n_hits, c->row_ptr, c->n_edges, s, c->flags);
  if (n_hits == 0) return;
  if (c->hp.k > 16) {
    const size_t n = (size_t)n_hits * 16;
    pack_edges_sparse_kernel<<<(unsigned)((n + 255) / 256), 256, 0, s>>>(c->nbr, c->deg, c->row_ptr, n_hits, c->hp.k, c->src, c->dst, c->flags);
  } else {
    const size_t n = (size_t)n_hits * c->hp.k;
    pack_edges_kernel<<<(unsigned)((n + 255) / 256), 256, 0, s>>>(c->nbr, c->deg, c->row_ptr, n_hits, c->hp.k, c->src, c->dst, c->flags);
  }
  c->launches++;
}

// injected, src-sorted edge list: row_ptr[q] = lower bound of q in src
__global__ void rows_from_src_kernel(const int32_t* __restrict__ src, int n_edges, int n_hits, int32_t* __restrict__ row_ptr) {
  int q = blockIdx.x * blockDim.x + threadIdx.x;
  if (q > n_hits) return;
  int lo = 0, hi = n_edges;
  while (lo < hi) { int mid = (lo + hi) >> 1; if (src[mid] < q) lo = mid + 1; else hi = mid; }
  row_ptr[q] = lo;
}

void launch_rows_from_src(etx_ctx* c, int n_hits, int n_edges, cudaStream_t s) {
  rows_from_src_kernel<<<(n_hits + 1 + 255) / 256, 256, 0, s>>>(c->src, n_edges, n_hits, c->row_ptr);
  c->launches++;
}

__global__ void indegree_kernel(const int32_t* __restrict__ dst, const int32_t* __restrict__ n_edges, int32_t* __restrict__ indeg) {
  const int E = *n_edges;
  for (int i = blockIdx.x * blockDim.x + threadIdx.x; i < E; i += gridDim.x * blockDim.x) atomicAdd(&indeg[dst[i]], 1);
}

__global__ void csc_fill_kernel(const int32_t* __restrict__ dst, const int32_t* __restrict__ n_edges,
                                int32_t* __restrict__ cursor, int32_t* __restrict__ in_edge) {
  const int E = *n_edges;
  for (int i = blockIdx.x * blockDim.x + threadIdx.x; i < E; i += gridDim.x * blockDim.x)
    in_edge[atomicAdd(&cursor[dst[i]], 1)] = i;
}

// ascending edge id inside every dst group (R9 / R22): groups are short (in-degree ~ k), insertion sort
__global__ void csc_sort_kernel(const int32_t* __restrict__ col_ptr, int n_hits, int32_t* __restrict__ in_edge) {
  int l = blockIdx.x * blockDim.x + threadIdx.x;
  if (l >= n_hits) return;
  const int a = col_ptr[l], b = col_ptr[l + 1];
  for (int i = a + 1; i < b; ++i) {
    int v = in_edge[i], j = i - 1;
    while (j >= a && in_edge[j] > v) { in_edge[j + 1] = in_edge[j]; --j; }
    in_edge[j + 1] = v;
  }
}

// Stable fill of one (event, plane) bucket of dst hits per WARP -- no sort.  Edges are sorted by src and a k-NN edge
// goes from plane q to a plane in q+1 .. q+w (R7, R25), so every in-edge of a hit on plane p lies in the contiguous
// edge range of the src planes p-w .. p-1 of the same event.  The warp walks that range in ascending edge id, 32
// edges per step (coalesced src / dst reads, eight steps loaded at once).  The neighbours of one src are distinct,
// so two lanes of a step can only meet on a dst if they belong to different src hits: the step is split into
// phases, one per src it spans (at most a handful), and in a phase every lane of that src advances its dst's
// cursor with a plain read-modify-write.  Phases and steps are sequential, so every dst group comes out in
// ascending edge id (R9 / R22) by construction.  A __syncwarp() separates them (shuffles and
// reductions are no memory barrier).  (match.any would rank the lanes of a step in one go, but costs
// ~1,400 cycles a step on this part.)  The cursors of a bucket are touched by this warp only (in shared memory, or
// in the global scratch `cursor` for a bucket of more than kCscHits hits; initialised from col_ptr), so there is no
// capacity limit and no atomic.
constexpr int kCscWarps = 8;
constexpr int kCscAhead = 8;                         // steps of 32 edges whose dst values are loaded together
constexpr int kCscHits = 1024;                       // cursors per warp in shared memory (4 KB)

__global__ void __launch_bounds__(kCscWarps * 32)
csc_bucket_kernel(const int32_t* __restrict__ src, const int32_t* __restrict__ dst, const int32_t* __restrict__ row_ptr,
                  const int32_t* __restrict__ col_ptr, const int32_t* __restrict__ plane_off, int n_buckets, int P, int w, int32_t* cursor, int32_t* __restrict__ in_edge) {
  const int bucket = blockIdx.x * kCscWarps + (threadIdx.x >> 5), lane = threadIdx.x & 31;
  if (bucket >= n_buckets) return;
  const int e = bucket / P, p = bucket % P;
  const int32_t* po = plane_off + (size_t)e * (P + 1);
  const int h0 = po[p], n = po[p + 1] - h0;
  if (n == 0) return;
  if (col_ptr[h0 + n] == col_ptr[h0]) return;                       // no in-edges at all
  const int q_lo = p - w > 0 ? p - w : 0;
  const int e0 = row_ptr[po[q_lo]], e1 = row_ptr[h0];               // out-edges of the src planes p-w .. p-1
  __shared__ int32_t cur_s[kCscWarps][kCscHits];
  volatile int32_t* cur = n <= kCscHits ? cur_s[threadIdx.x >> 5] : cursor + h0;   // shared unless the bucket is huge
  for (int i = lane; i < n; i += 32) cur[i] = col_ptr[h0 + i];
  __syncwarp();
  // The walk is sequential, so its speed is one global-load latency per batch of dst values: kCscAhead steps
  // (32 edges each) are loaded at once, then ranked and placed one after the other.
  for (int i0 = e0; i0 < e1; i0 += 32 * kCscAhead) {
    int dq[kCscAhead], sq[kCscAhead];
#pragma unroll
    for (int u = 0; u < kCscAhead; ++u) {
      const int i = i0 + 32 * u + lane;
      dq[u] = i < e1 ? dst[i] : -1;
      sq[u] = i < e1 ? src[i] : 0x7fffffff;
    }
#pragma unroll
    for (int u = 0; u < kCscAhead; ++u) {
      const int i = i0 + 32 * u + lane;
      if (i0 + 32 * u >= e1) break;                                  // warp-uniform
      const unsigned d = (unsigned)(dq[u] - h0);                     // -1 - h0 wraps above n
      const bool mine = dq[u] >= 0 && d < (unsigned)n;
      unsigned s_now = (unsigned)__shfl_sync(0xffffffffu, sq[u], 0);
      while (s_now < 0x7fffffffu) {                                  // one phase per src hit the step spans
        if (mine && (unsigned)sq[u] == s_now) { const int pos = cur[d]; cur[d] = pos + 1; in_edge[pos] = i; }
        __syncwarp();                                                // the next phase (or step) reads these cursors
        s_now = __reduce_min_sync(0xffffffffu, (unsigned)sq[u] > s_now ? (unsigned)sq[u] : 0x7fffffffu);
      }
    }
  }
}

// `windowed`: the edge list was built by S2 (every edge spans 1..w planes); an injected list takes the general path
void launch_csc(etx_ctx* c, int n_events, int n_hits, bool windowed, cudaStream_t s) {
  if (n_hits == 0) { exclusive_scan(c, c->cursor, 0, c->col_ptr, nullptr, s); return; }
  cudaMemsetAsync(c->cursor, 0, sizeof(int32_t) * ((size_t)n_hits + 1), s);
  const int grid = c->sm_count * 8;
  indegree_kernel<<<grid, 256, 0, s>>>(c->dst, c->n_edges, c->cursor);
  exclusive_scan(c, c->cursor, n_hits, c->col_ptr, nullptr, s);
  if (windowed && n_events > 0) {
    const int nb = n_events * c->hp.n_planes;
    csc_bucket_kernel<<<(nb + kCscWarps - 1) / kCscWarps, kCscWarps * 32, 0, s>>>(c->src, c->dst, c->row_ptr, c->col_ptr, c->plane_off, nb,
                                                                                c->hp.n_planes, c->hp.window, c->cursor, c->in_edge);
    c->launches += 2;
    return;
  }
  cudaMemcpyAsync(c->cursor, c->col_ptr, sizeof(int32_t) * (size_t)n_hits, cudaMemcpyDeviceToDevice, s);
  csc_fill_kernel<<<grid, 256, 0, s>>>(c->dst, c->n_edges, c->cursor, c->in_edge);
  csc_sort_kernel<<<(n_hits + 255) / 256, 256, 0, s>>>(c->col_ptr, n_hits, c->in_edge);
  c->launches += 3;
}

// --------------------------------------------------------------------------------------------------------
// S5 (L80, L82, L206, L261 sec. 7.3; R17, R18): an edge is kept iff logit >= tau; track_id[h] = smallest hit
// index in h's component of the kept-edge graph.  The paper's kernel propagates the lowest label with one
// forward and one backward plane sweep (a heuristic that can under-merge); here exact components by a
// lock-free union-find: a root is only ever re-pointed to a SMALLER index, so the final root of a set is
// its minimum and the result does not depend on the interleaving.  Pointer jumping compresses paths.
__device__ __forceinline__ int uf_find(int32_t* parent_, int x) {
  volatile int32_t* parent = parent_;  // other threads re-point entries concurrently: always re-read
  int p = parent[x];
  while (p != x) {
    int gp = parent[p];
    if (gp != p) parent[x] = gp;       // path halving (benign race: only ever stores an ancestor)
    x = p; p = gp;
  }
  return x;
}

// hang the root of one endpoint's set under the root of the other; `par` may be shared or global memory
__device__ __forceinline__ void uf_union(int32_t* par, int a, int b) {
  a = uf_find(par, a); b = uf_find(par, b);
  while (a != b) {
    if (a > b) { int t = a; a = b; b = t; }         // a < b : hang root b under a
    int old = atomicCAS(&par[b], b, a);
    if (old == b) break;
    b = uf_find(par, old);                          // b was no longer a root: retry from its new root
    a = uf_find(par, a);
  }
}

// Components never cross an event (R8), so one CTA labels one event with its parent array in shared memory
// (local hit indices; the paper's per-event smem labelling, L261, made exact).  The event's edges are the
// contiguous range row_ptr[first hit] .. row_ptr[end hit) because edges are sorted by src (R9); src, dst and
// logit are read once, coalesced.  Events with more hits than the shared array use their slice of the global
// output as the parent array, with the same code.
constexpr int kUfThreads = 1024;
constexpr int kUfSmemHits = 16384;                  // 64 KB

__global__ void __launch_bounds__(kUfThreads)
uf_event_kernel(const int32_t* __restrict__ src, const int32_t* __restrict__ dst, const float* __restrict__ logit,
                const int32_t* __restrict__ row_ptr, const int32_t* __restrict__ event_off, int n_events, float tau,
                int32_t* track_id) {
  extern __shared__ int32_t uf_smem[];
  for (int e = blockIdx.x; e < n_events; e += gridDim.x) {
    const int h0 = event_off[e], n = event_off[e + 1] - h0;
    if (n <= 0) continue;
    const int e0 = row_ptr[h0], e1 = row_ptr[h0 + n];
    const bool in_smem = n <= kUfSmemHits;
    int32_t* par = in_smem ? uf_smem : track_id + h0;
    for (int i = threadIdx.x; i < n; i += kUfThreads) par[i] = i;
    __syncthreads();
    // the three streams are read one iteration ahead: the loop body (finds, CAS) depends on them, and an edge per
    // ~1 us of load latency per thread is what this kernel would otherwise run at
    int i = e0 + threadIdx.x;
    float z = 0.0f; int s_ = 0, d_ = 0;
    if (i < e1) { z = logit[i]; s_ = src[i]; d_ = dst[i]; }
    while (i < e1) {
      const float zc = z; const int sc = s_, dc = d_;
      i += kUfThreads;
      if (i < e1) { z = logit[i]; s_ = src[i]; d_ = dst[i]; }
      if (!(zc >= tau)) continue;                   // R17: kept iff z >= tau
      const unsigned a = (unsigned)(sc - h0), b = (unsigned)(dc - h0);
      if (a >= (unsigned)n || b >= (unsigned)n) continue;   // cannot happen for edges built by S2 (R8)
      uf_union(par, (int)a, (int)b);
    }
    __syncthreads();
    if (in_smem) {
      for (int i = threadIdx.x; i < n; i += kUfThreads) {
        int r = i;
        while (true) { const int p = par[r]; if (p == r) break; r = p; }
        track_id[h0 + i] = h0 + r;
      }
    } else {
      volatile int32_t* vp = par;
      for (int i = threadIdx.x; i < n; i += kUfThreads) {
        int r = i;
        while (true) { const int p = vp[r]; if (p == r) break; r = p; }
        vp[i] = r;                                  // racing readers still see an ancestor of i
      }
      __syncthreads();
      for (int i = threadIdx.x; i < n; i += kUfThreads) par[i] += h0;
    }
    __syncthreads();
  }
}

void launch_components(etx_ctx* c, const float* logit, int n_events, int n_hits, cudaStream_t s) {
  if (n_hits == 0 || n_events == 0) return;
  constexpr int smem = kUfSmemHits * (int)sizeof(int32_t);
  opt_in_smem(c, uf_event_kernel, smem);
  const int grid = n_events;                          // one CTA per event; the hardware balances them
  uf_event_kernel<<<grid, kUfThreads, smem, s>>>(c->src, c->dst, logit, c->row_ptr, c->event_off, n_events, c->tau, c->track_id);
  c->launches += 1;
}

// --------------------------------------------------------------------------------------------------------
// Track containers (reconstructible = at least three hits; L74, L82: the pipeline's product is the
// set of tracks, each a list of hits).  A track is a component with >= min_hits hits;
// tracks are numbered densely in ascending order of their root (= smallest hit index = track_id), so the tracks
// of an event are consecutive; hits inside a track ascend.
__global__ void trk_size_kernel(const int32_t* __restrict__ track_id, int n, int32_t* __restrict__ size) {
  const int h = blockIdx.x * blockDim.x + threadIdx.x;
  if (h < n) atomicAdd(&size[track_id[h]], 1);
}
__global__ void trk_keep_kernel(const int32_t* __restrict__ track_id, const int32_t* __restrict__ size, int n, int min_hits,
                                int32_t* __restrict__ keep) {
  const int r = blockIdx.x * blockDim.x + threadIdx.x;
  if (r < n) keep[r] = (track_id[r] == r && size[r] >= min_hits) ? 1 : 0;
}
// number[r] = exclusive scan of keep: dense number of root r.  Sizes of the kept tracks in dense order, and per hit
// the dense number of its track (or -1).
__global__ void trk_index_kernel(const int32_t* __restrict__ track_id, const int32_t* __restrict__ size,
                                 const int32_t* __restrict__ number, int n, int min_hits,
                                 int32_t* __restrict__ track_index, int32_t* __restrict__ ksize) {
  const int h = blockIdx.x * blockDim.x + threadIdx.x;
  if (h >= n) return;
  const int r = track_id[h];
  const bool kept = size[r] >= min_hits;
  track_index[h] = kept ? number[r] : -1;
  if (kept && r == h) ksize[number[r]] = size[r];
}
__global__ void trk_event_kernel(const int32_t* __restrict__ event_off, const int32_t* __restrict__ number, int n_events,
                                 int32_t* __restrict__ event_track_off) {
  const int e = blockIdx.x * blockDim.x + threadIdx.x;
  if (e <= n_events) event_track_off[e] = number[event_off[e]];
}
// One warp per event walks the event's hits in ascending order, 32 per step; the lanes of a step that share a track
// are ranked with match.any and the lowest advances the track's cursor, so every hit list ascends by construction.
// The cursors of an event's tracks are touched by this warp only.
__global__ void __launch_bounds__(256)
trk_fill_kernel(const int32_t* __restrict__ track_index, const int32_t* __restrict__ track_offsets,
                const int32_t* __restrict__ event_off, const int32_t* __restrict__ event_track_off, int n_events,
                int32_t* cursor, int32_t* __restrict__ track_hits) {
  const int e = blockIdx.x * 8 + (threadIdx.x >> 5), lane = threadIdx.x & 31;
  if (e >= n_events) return;
  const int h0 = event_off[e], h1 = event_off[e + 1];
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

void launch_tracks(etx_ctx* c, int n_events, int n_hits, int min_hits, cudaStream_t s) {
  cudaMemsetAsync(c->n_tracks, 0, sizeof(int32_t), s);
  if (n_hits == 0 || n_events == 0) {
    cudaMemsetAsync(c->trk_event_off, 0, sizeof(int32_t) * ((size_t)n_events + 1), s);
    cudaMemsetAsync(c->trk_offsets, 0, sizeof(int32_t), s);
    return;
  }
  const int g = (n_hits + 255) / 256;
  cudaMemsetAsync(c->trk_size, 0, sizeof(int32_t) * (size_t)n_hits, s);
  cudaMemsetAsync(c->trk_ksize, 0, sizeof(int32_t) * (size_t)n_hits, s);
  trk_size_kernel<<<g, 256, 0, s>>>(c->track_id, n_hits, c->trk_size);
  trk_keep_kernel<<<g, 256, 0, s>>>(c->track_id, c->trk_size, n_hits, min_hits, c->trk_keep);
  exclusive_scan(c, c->trk_keep, n_hits, c->trk_number, c->n_tracks, s);
  trk_index_kernel<<<g, 256, 0, s>>>(c->track_id, c->trk_size, c->trk_number, n_hits, min_hits, c->trk_index, c->trk_ksize);
  exclusive_scan(c, c->trk_ksize, n_hits, c->trk_offsets, nullptr, s);       // entries >= n_tracks repeat the total
  trk_event_kernel<<<(n_events + 256) / 256, 256, 0, s>>>(c->event_off, c->trk_number, n_events, c->trk_event_off);
  trk_fill_kernel<<<(n_events + 7) / 8, 256, 0, s>>>(c->trk_index, c->trk_offsets, c->event_off, c->trk_event_off, n_events,
                                                     c->trk_keep, c->trk_hits);      // trk_keep is free again: cursors
  c->launches += 5;
}

// --------------------------------------------------------------------------------------------------------
// Triplet building (sec. 5.3; R29) on the purified hit graph (edges with logit >= tau, L80).
// A triplet is a pair of kept edges (first, second) with one common hit C: kind 0 articulation (an in-edge and an
// out-edge of C), kind 1 left elbow (two out-edges of C), kind 2 right elbow (two in-edges of C), first < second for
// the elbows.  Order: C ascending, then first, then second -- which is the order of the CSR / CSC lists, both
// ascending in edge id.  Count per hit -> exclusive scan -> fill; all integer work, bit-exact by construction.
// Counts, offsets and totals of triplets are int32 and SATURATE at kTripSat = 2^31 - 1 instead of wrapping (threshold
// near 0, large k and a large batch can exceed it): a saturated offset is >= any capacity, so nothing is written for it,
// and a total of 2^31 - 1 reads "at least that many".  Saturating addition of non-negative numbers is associative, so
// the block-wise prefix sum below is exact up to the limit.  (S3's own scan stays the plain one: E <= k * max_hits.)
constexpr int32_t kTripSat = 0x7fffffff;
__device__ __forceinline__ int sat_add(int a, int b) {          // a, b in [0, kTripSat]
  const unsigned s = (unsigned)a + (unsigned)b;
  return s > (unsigned)kTripSat ? kTripSat : (int)s;
}
// exclusive saturating prefix sum of one value per thread over the block (blockDim = kScanThreads); *total = block sum
__device__ __forceinline__ int block_exclusive_sat_scan(int v, int* total) {
  __shared__ int warp_incl[kScanThreads / 32];
  const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
  int x = v;
#pragma unroll
  for (int o = 1; o < 32; o <<= 1) { const int y = __shfl_up_sync(0xffffffffu, x, o); if (lane >= o) x = sat_add(x, y); }
  int excl = __shfl_up_sync(0xffffffffu, x, 1);                 // the exclusive value is shuffled, not "inclusive - v"
  if (lane == 0) excl = 0;
  if (lane == 31) warp_incl[wid] = x;
  __syncthreads();
  int base = 0, all = 0;
#pragma unroll
  for (int i = 0; i < kScanThreads / 32; ++i) { const int s = warp_incl[i]; if (i < wid) base = sat_add(base, s); all = sat_add(all, s); }
  __syncthreads();
  *total = all;
  return sat_add(base, excl);
}
__global__ void __launch_bounds__(kScanThreads) sat_scan_reduce_kernel(const int32_t* __restrict__ in, int n, int32_t* __restrict__ bsum) {
  const int base = blockIdx.x * kScanChunk;
  int v = 0;
#pragma unroll
  for (int j = 0; j < kScanItems; ++j) { const int i = base + threadIdx.x * kScanItems + j; if (i < n) v = sat_add(v, in[i]); }
  int tot; block_exclusive_sat_scan(v, &tot);
  if (threadIdx.x == 0) bsum[blockIdx.x] = tot;
}
__global__ void __launch_bounds__(kScanThreads) sat_scan_bsum_kernel(int32_t* __restrict__ bsum, int nb) {
  int carry = 0;                                   // single block, sequential over chunks of 256
  for (int b0 = 0; b0 < nb; b0 += kScanThreads) {
    const int i = b0 + threadIdx.x;
    int tot;
    const int ex = block_exclusive_sat_scan(i < nb ? bsum[i] : 0, &tot);
    if (i < nb) bsum[i] = sat_add(carry, ex);
    carry = sat_add(carry, tot);
  }
}
__global__ void __launch_bounds__(kScanThreads) sat_scan_write_kernel(const int32_t* __restrict__ in, int n, const int32_t* __restrict__ bsum,
                                                                     int32_t* __restrict__ out) {
  const int base = blockIdx.x * kScanChunk;
  int vals[kScanItems], v = 0;
#pragma unroll
  for (int j = 0; j < kScanItems; ++j) {
    const int i = base + threadIdx.x * kScanItems + j;
    vals[j] = i < n ? in[i] : 0;
    v = sat_add(v, vals[j]);
  }
  int tot;
  int ex = sat_add(block_exclusive_sat_scan(v, &tot), bsum[blockIdx.x]);
#pragma unroll
  for (int j = 0; j < kScanItems; ++j) {
    const int i = base + threadIdx.x * kScanItems + j;
    if (i < n) out[i] = ex;
    ex = sat_add(ex, vals[j]);
    if (i == n - 1) out[n] = ex;
  }
}
// out[0..n] = exclusive saturating prefix sums of in[0..n), n >= 1
static void exclusive_sat_scan(etx_ctx* c, const int32_t* in, int n, int32_t* out, cudaStream_t s) {
  const int nb = (n + kScanChunk - 1) / kScanChunk;
  sat_scan_reduce_kernel<<<nb, kScanThreads, 0, s>>>(in, n, c->scan_tmp);
  sat_scan_bsum_kernel<<<1, kScanThreads, 0, s>>>(c->scan_tmp, nb);
  sat_scan_write_kernel<<<nb, kScanThreads, 0, s>>>(in, n, c->scan_tmp, out);
  c->launches += 3;
}

__global__ void trip_count_kernel(const int32_t* __restrict__ row_ptr, const int32_t* __restrict__ col_ptr,
                                  const int32_t* __restrict__ in_edge, const float* __restrict__ logit, float tau, int n_hits,
                                  int32_t* __restrict__ cnt /* [3][n_hits + 1] */) {
  const int c = blockIdx.x * blockDim.x + threadIdx.x;
  if (c >= n_hits) return;
  int od = 0, id = 0;
  for (int i = row_ptr[c]; i < row_ptr[c + 1]; ++i) od += logit[i] >= tau;
  for (int i = col_ptr[c]; i < col_ptr[c + 1]; ++i) id += logit[in_edge[i]] >= tau;
  const size_t st = (size_t)n_hits + 1;
  const long long lid = id, lod = od;                           // an in-degree of 65,536 already overflows id * (id - 1) in 32 bits
  cnt[c] = (int32_t)min(lid * lod, (long long)kTripSat);
  cnt[st + c] = (int32_t)min(lod * (lod - 1) / 2, (long long)kTripSat);
  cnt[2 * st + c] = (int32_t)min(lid * (lid - 1) / 2, (long long)kTripSat);
}

// one thread per common hit; triplets beyond `cap` are counted but not written (the caller compares the totals)
__global__ void trip_fill_kernel(const int32_t* __restrict__ row_ptr, const int32_t* __restrict__ col_ptr,
                                 const int32_t* __restrict__ in_edge, const float* __restrict__ logit, float tau, int n_hits,
                                 const int32_t* __restrict__ off /* [3][n_hits + 1] */, int cap,
                                 int32_t* __restrict__ first, int32_t* __restrict__ second, int32_t* __restrict__ hit /* [3][cap] */) {
  const int c = blockIdx.x * blockDim.x + threadIdx.x;
  if (c >= n_hits) return;
  const size_t st = (size_t)n_hits + 1;
  const int a0 = row_ptr[c], a1 = row_ptr[c + 1], b0 = col_ptr[c], b1 = col_ptr[c + 1];
  auto put = [&](int kind, int pos, int f, int s2) {
    if (pos >= 0 && pos < cap) { const size_t o = (size_t)kind * cap + pos; first[o] = f; second[o] = s2; hit[o] = c; }
  };
  auto next = [](int& p) { const int q = p; if (p < kTripSat) ++p; return q; };     // a saturated offset stays saturated
  int pa = off[c], pl = off[st + c], pr = off[2 * st + c];
  for (int i = b0; i < b1; ++i) {                               // in-edges of c, ascending edge id
    const int ei = in_edge[i];
    if (!(logit[ei] >= tau)) continue;
    for (int j = a0; j < a1; ++j) if (logit[j] >= tau) put(0, next(pa), ei, j);              // articulations
    for (int j = i + 1; j < b1; ++j) { const int ej = in_edge[j]; if (logit[ej] >= tau) put(2, next(pr), ei, ej); }   // right elbows
  }
  for (int i = a0; i < a1; ++i) {                               // out-edges of c
    if (!(logit[i] >= tau)) continue;
    for (int j = i + 1; j < a1; ++j) if (logit[j] >= tau) put(1, next(pl), i, j);            // left elbows
  }
}

__global__ void trip_totals_kernel(const int32_t* __restrict__ off, int n_hits, int32_t* __restrict__ total) {
  if (threadIdx.x < 3) total[threadIdx.x] = off[(size_t)threadIdx.x * ((size_t)n_hits + 1) + n_hits];
}

void launch_triplet_build(etx_ctx* c, int n_hits, cudaStream_t s) {
  if (n_hits == 0) { cudaMemsetAsync(c->trip_total, 0, 3 * sizeof(int32_t), s); return; }
  const int g = (n_hits + 127) / 128;
  const size_t st = (size_t)n_hits + 1;
  trip_count_kernel<<<g, 128, 0, s>>>(c->row_ptr, c->col_ptr, c->in_edge, c->logit, c->tau, n_hits, c->trip_cnt);
  for (int k = 0; k < 3; ++k) exclusive_sat_scan(c, c->trip_cnt + k * st, n_hits, c->trip_off + k * st, s);
  trip_totals_kernel<<<1, 32, 0, s>>>(c->trip_off, n_hits, c->trip_total);
  trip_fill_kernel<<<g, 128, 0, s>>>(c->row_ptr, c->col_ptr, c->in_edge, c->logit, c->tau, n_hits, c->trip_off, c->hp.max_triplets,
                                     c->trip_first, c->trip_second, c->trip_hit);
  c->launches += 3;
}

// --------------------------------------------------------------------------------------------------------
// Track building from triplets, phases (1)-(2) (sec. 5.4; R30): which kept edges end up
// in one set of connected edges, and which articulations are shared.  Same lock-free union-find as S5 (roots only
// ever move to a smaller index, so a set is named by its smallest edge id whatever the interleaving); the distinct
// (super-edge, super-edge) articulation pairs are collected in an open-addressing hash set, the first inserter of a
// pair counting it as a successor / predecessor.  All outputs are sets or minima: deterministic.
constexpr unsigned long long kTcEmpty = 0xffffffffffffffffull;

__global__ void tc_init_kernel(int32_t* __restrict__ par1, int32_t* __restrict__ par2, int32_t* __restrict__ n_succ,
                               int32_t* __restrict__ n_pred, const int32_t* __restrict__ n_edges,
                               unsigned long long* __restrict__ tab, size_t tab_size, int32_t* __restrict__ n_shared) {
  const int E = *n_edges;
  const size_t stride = (size_t)gridDim.x * blockDim.x, t0 = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
  for (size_t i = t0; i < (size_t)E; i += stride) { par1[i] = (int32_t)i; par2[i] = (int32_t)i; n_succ[i] = 0; n_pred[i] = 0; }
  for (size_t i = t0; i < tab_size; i += stride) tab[i] = kTcEmpty;
  if (t0 == 0) *n_shared = 0;
}

// (1) the two edges of every kept elbow (kinds 1 and 2) become one super-edge
__global__ void tc_elbows_kernel(const int32_t* __restrict__ first, const int32_t* __restrict__ second, const float* __restrict__ logit,
                                 const int32_t* __restrict__ total, int cap, float tau_t, int32_t* par1) {
  const size_t stride = (size_t)gridDim.x * blockDim.x;
  for (int kind = 1; kind <= 2; ++kind) {
    const int n = max(0, min(total[kind], cap));
    const size_t o = (size_t)kind * cap;
    for (size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x; i < (size_t)n; i += stride)
      if (logit[o + i] >= tau_t) uf_union(par1, first[o + i], second[o + i]);
  }
}

__device__ __forceinline__ size_t tc_hash(unsigned long long k, size_t mask) {
  k ^= k >> 33; k *= 0xff51afd7ed558ccdull; k ^= k >> 33; k *= 0xc4ceb9fe1a85ec53ull; k ^= k >> 33;
  return (size_t)k & mask;
}

// kept articulations mapped onto super-edges; duplicates collapse, one inside a super-edge disappears
__global__ void tc_arts_kernel(const int32_t* __restrict__ first, const int32_t* __restrict__ second, const float* __restrict__ logit,
                               const int32_t* __restrict__ total, int cap, float tau_t, int32_t* par1,
                               unsigned long long* tab, size_t mask, int32_t* n_succ, int32_t* n_pred) {
  const int n = max(0, min(total[0], cap));
  const size_t stride = (size_t)gridDim.x * blockDim.x;
  for (size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x; i < (size_t)n; i += stride) {
    if (!(logit[i] >= tau_t)) continue;
    const int x = uf_find(par1, first[i]), y = uf_find(par1, second[i]);
    if (x == y) continue;
    const unsigned long long key = ((unsigned long long)(unsigned)x << 32) | (unsigned)y;
    size_t slot = tc_hash(key, mask);
    while (true) {
      const unsigned long long old = atomicCAS(&tab[slot], kTcEmpty, key);
      if (old == kTcEmpty) { atomicAdd(&n_succ[x], 1); atomicAdd(&n_pred[y], 1); break; }
      if (old == key) break;
      slot = (slot + 1) & mask;
    }
  }
}

// (2) a pair is shared iff its first super-edge has >= 2 distinct successors or its second >= 2 distinct predecessors;
// the others connect their super-edges
__global__ void tc_link_kernel(const unsigned long long* __restrict__ tab, size_t tab_size, const int32_t* __restrict__ n_succ,
                               const int32_t* __restrict__ n_pred, int32_t* par2, int32_t* __restrict__ shared, int32_t* n_shared, int cap) {
  const size_t stride = (size_t)gridDim.x * blockDim.x;
  for (size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x; i < tab_size; i += stride) {
    const unsigned long long key = tab[i];
    if (key == kTcEmpty) continue;
    const int x = (int)(key >> 32), y = (int)(key & 0xffffffffu);
    if (n_succ[x] >= 2 || n_pred[y] >= 2) {
      const int p = atomicAdd(n_shared, 1);
      if (p < cap) { shared[2 * (size_t)p] = x; shared[2 * (size_t)p + 1] = y; }
    } else {
      uf_union(par2, x, y);
    }
  }
}

__global__ void tc_label_kernel(const float* __restrict__ edge_logit, float tau, const int32_t* __restrict__ n_edges, int32_t* par1,
                                int32_t* par2, int32_t* __restrict__ edge_comp, int32_t* __restrict__ shared,
                                const int32_t* __restrict__ n_shared, int cap) {
  const int E = *n_edges, ns = max(0, min(*n_shared, cap));
  const size_t stride = (size_t)gridDim.x * blockDim.x, t0 = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
  for (size_t i = t0; i < (size_t)E; i += stride) edge_comp[i] = edge_logit[i] >= tau ? uf_find(par2, uf_find(par1, (int)i)) : -1;
  for (size_t i = t0; i < 2 * (size_t)ns; i += stride) shared[i] = uf_find(par2, shared[i]);
}

void launch_triplet_components(etx_ctx* c, cudaStream_t s) {
  const int g = c->sm_count * 8, cap = c->hp.max_triplets;
  tc_init_kernel<<<g, 256, 0, s>>>(c->tc_par1, c->tc_par2, c->tc_succ, c->tc_pred, c->n_edges, c->tc_tab, c->tc_tab_size, c->tc_n_shared);
  tc_elbows_kernel<<<g, 256, 0, s>>>(c->trip_first, c->trip_second, c->trip_logit, c->trip_total, cap, c->tau_t, c->tc_par1);
  tc_arts_kernel<<<g, 256, 0, s>>>(c->trip_first, c->trip_second, c->trip_logit, c->trip_total, cap, c->tau_t, c->tc_par1,
                                   c->tc_tab, c->tc_tab_size - 1, c->tc_succ, c->tc_pred);
  tc_link_kernel<<<g, 256, 0, s>>>(c->tc_tab, c->tc_tab_size, c->tc_succ, c->tc_pred, c->tc_par2, c->tc_shared, c->tc_n_shared, cap);
  tc_label_kernel<<<g, 256, 0, s>>>(c->logit, c->tau, c->n_edges, c->tc_par1, c->tc_par2, c->tc_comp, c->tc_shared, c->tc_n_shared, cap);
  c->launches += 5;
}

}  // namespace etx
