/* ============================================================================
 * etx.h -- C-ABI boundary of the B200-native ETX4VELO hot path.
 *
 * The path (sec. 7: "embedding inference, k-NN, GNN up to the edge
 * classifier, WCC"; triplet steps excluded exactly as in the paper's CUDA code,
 * L20 / L238), batched over many events (L12 abstract, L38 sec. 2, L223 sec. 7:
 * 500 events per stream):
 *
 *   S0 plane offsets      hits arrive per (event, plane)              L26, L223, L257
 *   S1 embedding MLP      e_h = MLP(norm(x,y,z))                      L96 sec. 5.1, L107 fn.5
 *   S2 k-NN               k nearest hits on planes p+1..p+w, d2<d2max L98 Eq.(1), L101, L257 sec. 7.2
 *   S3 edge list          G_rough^hit, directed i->j, i on lower plane L74-76, L137
 *   S4 interaction net    encoders, L x (Eq.(4) messages, node net,
 *                         edge net, residual), edge classifier        L133-148 sec. 5.2
 *   S5 threshold + WCC    discard score < s_edge,min; components      L80, L82, L206, L261 sec. 7.3
 *   (separate calls, not part of the timed path: etx_tracks -- track containers, L42 / L74 / L82;
 *    etx_triplets, etx_triplet_components, etx_triplet_tracks -- the triplet stage, L150-176 sec. 5.3-5.4)
 *
 * Readings of every point where the paper is silent are in DESIGN.md sec. 4
 * (R1..R31).  All pointers are plain pointers; "d_" = device memory on the
 * current CUDA device, "h_" = host memory.  No C++ or torch types cross this
 * boundary.  Every function returns an etx_status; nothing throws across the boundary.  One device-side guard
 * exists: a kernel that waits more than ~20 s of wall-clock time on one mbarrier (a lost arrival, i.e. a bug)
 * executes a trap instead of hanging the GPU, which surfaces as ETX_ERR_CUDA on the next call.
 * ==========================================================================*/
#ifndef ETX_H_
#define ETX_H_

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct etx_ctx* etx_handle;
typedef void* etx_stream;            /* a cudaStream_t, passed as an opaque pointer (NULL = default stream) */

typedef enum {
  ETX_OK = 0,
  ETX_ERR_ARG = -1,          /* null pointer, negative size, inconsistent offsets            */
  ETX_ERR_BLOB = -2,         /* weights blob: bad magic / version / shapes / size / scales   */
  ETX_ERR_CAPACITY = -3,     /* n_events > max_events or n_hits > max_hits                   */
  ETX_ERR_INPUT_ORDER = -4,  /* device-side validation found hits not sorted by (event,plane),
                                or a plane index outside [0, n_planes): see etx_input_status  */
  ETX_ERR_CUDA = -5,         /* a CUDA runtime call failed; see etx_last_error               */
  ETX_ERR_UNSUPPORTED = -6   /* shape / precision not built into this library                */
} etx_status;

typedef enum { ETX_FP32 = 0, ETX_BF16 = 1, ETX_INT8 = 2 } etx_precision;

/* Storage of the GNN state h, e, m (R20 / R21).  AUTO: fp32 for ETX_FP32 and ETX_INT8,
 * bf16 for ETX_BF16.  ETX_INT8 may also store it in bf16 (RNE on store, fp32 arithmetic on the widened values): half
 * the HBM bytes of the S4 loop.  Other combinations are ETX_ERR_UNSUPPORTED. */
typedef enum { ETX_STATE_AUTO = 0, ETX_STATE_FP32 = 1, ETX_STATE_BF16 = 2 } etx_state_dtype;

/* How the MLP layers with K >= 16 are executed (the K = 3 input layers and the d->1 head are
 * always fp32 FFMA in a pinned order, R4/R20/R21). */
typedef enum {
  ETX_ENGINE_AUTO = 0,       /* fp32: FFMA kernels; bf16 / int8: tcgen05 tensor-core kernels  */
  ETX_ENGINE_SIMT = 1,       /* FFMA kernels in every precision (bf16 / int8 rounding points
                                reproduced exactly; the deterministic debugging path)         */
  ETX_ENGINE_TC_SERIAL = 2   /* tensor-core kernels without warp specialisation (one tile at a
                                time per CTA); same arithmetic as AUTO, kept as a cross-check */
} etx_engine;

typedef struct {
  uint32_t struct_size;              /* sizeof(etx_hyperparams); ABI check                              */
  int32_t  n_planes;                 /* 26 (L26)                                                        */
  float    norm_offset[3];           /* f = (x + offset) / div, true IEEE division (L107 fn.5, R1)      */
  float    norm_div[3];
  int32_t  emb_hidden;               /* width D of the embedding MLP's hidden layers (64 | 128)         */
  int32_t  emb_n_hidden_layers;      /* H hidden layers: 3 -> D -> ... -> D -> emb_dim                  */
  int32_t  emb_dim;                  /* 4                                                               */
  int32_t  k;                        /* k_max neighbours per hit (L101)                                 */
  int32_t  window;                   /* w: candidates on planes p+1..p+w (L101: 2)                      */
  float    d2_max;                   /* keep candidate iff d2 < d2_max; +inf = no cut (L101, R6)        */
  int32_t  gnn_latent;               /* d = n_h = n_e (L148)                                            */
  int32_t  gnn_iters;                /* L message-passing steps with distinct weights (L148)            */
  int32_t  edge_enc_input;           /* 0: |f_dst - f_src| (BASELINE configs)  1: [h0_src,h0_dst] (L133)*/
  float    threshold;                /* s_edge,min: keep edge iff score >= threshold (L80, R17)         */
  int32_t  precision;                /* etx_precision of the MLP layers with K >= 16                    */
  int32_t  engine;                   /* etx_engine                                                      */
  int32_t  max_events;               /* workspace capacity (L223: fixed memory per stream)              */
  int32_t  max_hits;                 /* max_edges = k * max_hits                                        */
  int32_t  validate_input;           /* 1: device-side check that hits are sorted by (event, plane)     */
  int32_t  emb_input;                /* input of the embedding MLP.  0: the Cartesian features above (BASELINE
                                        configs)  1: ((r, phi, z) + cyl_offset) / cyl_div, the paper's normalised
                                        cylindrical coordinates (L96); r = sqrt(fma(y,y,x*x)), phi = the fp32
                                        polynomial atan2 of DESIGN.md R27 (|error| <= 5e-7).  Must equal word 10
                                        of the blob header.  The GNN encoders always read the Cartesian
                                        features (L133).                                                   */
  float    cyl_offset[3];
  float    cyl_div[3];
  int32_t  state_dtype;              /* etx_state_dtype                                                                  */
  int32_t  max_triplets;             /* capacity per triplet kind of etx_triplets (0: the triplet stage is not used)     */
  float    triplet_threshold;        /* a triplet is kept iff its score >= this (L80: "triplets scoring below ... are
                                        discarded"; decided on the logit like the edge threshold, R17)                  */
  /* Optional device-memory allocator (L223: Allen hands every algorithm memory from its own per-stream
   * arena).  NULL alloc: cudaMalloc / cudaFree.  alloc must return device memory aligned to 256 bytes or
   * NULL on failure; dealloc is called once per block from etx_destroy; alloc and dealloc go together.    */
  void*  (*alloc)(size_t bytes, void* alloc_ctx);
  void   (*dealloc)(void* ptr, void* alloc_ctx);
  void*  alloc_ctx;
} etx_hyperparams;

typedef struct {                     /* device pointers into the handle's workspace (library-owned);   */
  const int32_t* d_edge_src;         /* [n_edges]  valid until the next call on the handle             */
  const int32_t* d_edge_dst;         /* [n_edges]  edges ordered by (src asc, neighbour rank asc) (R9)  */
  const float*   d_edge_score;       /* [n_edges]  sigmoid of the edge classifier output (L80)          */
  const float*   d_edge_logit;       /* [n_edges]  pre-sigmoid value; the threshold is applied here     */
  const int32_t* d_track_id;         /* [n_hits]   smallest global hit index of the hit's component     */
  const int32_t* d_n_edges;          /* device scalar                                                   */
  const int32_t* h_n_edges;          /* pinned host mirror; valid once the stream has been synchronised */
  int32_t        n_hits;
} etx_output;

/* Create a context: parse + validate the weights blob (layout: datagen/weights.py header; fp32
 * tensors W[out][in], b[out] in the order emb 0..H, node enc (2), edge enc (2), per step node net (2)
 * + edge net (2), head, and -- if header word 11 is set -- the articulation and the elbow triplet classifier
 * (2d -> d, d -> 1 each); INT8 additionally one activation scale per Linear with K >= 16), convert the
 * weights to the precision's operand format, allocate the workspace for (max_events, max_hits, k).
 * The blob is copied; the caller may free it on return.  *out is set only on ETX_OK. */
etx_status etx_create(const void* h_weights_blob, size_t blob_bytes, const etx_hyperparams* hp,
                      etx_handle* out);

/* Enqueue the whole path S0..S5 for one packed batch on `stream` and return without synchronising the stream or
 * the device.  (The one host-side wait: the event offsets travel through a pinned staging buffer of the handle, and
 * the call blocks until the previous call's copy out of that buffer has been issued to the device -- microseconds.)
 * The CUDA device that was current at etx_create must be current (ETX_ERR_ARG otherwise).
 *   d_xyz             [n_hits][3] fp32, millimetres, device; borrowed until the enqueued work is done
 *   d_plane           [n_hits] int32 in [0, n_planes), device; hits sorted by (event, plane)
 *   h_event_offsets   [n_events+1] int32, host; [0] = 0, non-decreasing, [n_events] = n_hits
 * Empty events / planes are legal; n_events = 0 is a no-op that reports 0 edges.
 * One handle serves one stream at a time; calls on one handle are not thread-safe.
 * Input validation (hyperparams.validate_input = 1) runs on the device as part of S0.  A batch that breaks the
 * input contract is REJECTED on the device: its row offsets and edge count are forced to 0, so no later stage
 * touches memory on its behalf, n_edges = 0 and track_id[h] = h.  etx_run itself still returns ETX_OK (it cannot
 * know without synchronising); the verdict of the batch is read with etx_input_status after the stream has been
 * synchronised.  A rejected batch never affects the calls that follow it.  Without validate_input an out-of-contract
 * batch is the caller's responsibility (results undefined, memory accesses still bounded by the workspace). */
etx_status etx_run(etx_handle h, const float* d_xyz, const int32_t* d_plane,
                   const int32_t* h_event_offsets, int32_t n_events, etx_stream stream,
                   etx_output* out);

/* The same call with HOST buffers (the end-to-end measurement of bench.py): copies xyz / plane to the
 * device, runs S0..S5, copies edge_score [n_edges], edge_src/dst (if non-NULL) and track_id [n_hits]
 * back, and synchronises `stream`.  h_* output buffers must hold k*n_hits (edges) / n_hits entries.
 * Pinned host memory makes the copies asynchronous (src / dst are copied under the GNN, and the scores
 * are written by the classifier straight into a pinned h_edge_score, which is device-addressable);
 * pageable memory works too.  *n_edges_out = E. */
/* Returns ETX_ERR_INPUT_ORDER when validate_input is set and the batch was rejected (it synchronises anyway). */
etx_status etx_run_host(etx_handle h, const float* h_xyz, const int32_t* h_plane,
                        const int32_t* h_event_offsets, int32_t n_events, etx_stream stream,
                        float* h_edge_score, int32_t* h_edge_src, int32_t* h_edge_dst,
                        int32_t* h_track_id, int32_t* n_edges_out);

/* The same work as etx_run_host, asynchronously and pipelined (Allen keeps several streams of events
 * in flight so that copies hide under compute): etx_submit_host enqueues the H2D copy of the inputs (on the handle's
 * copy stream, under the previous batch's compute), S0..S5 on `stream`, and the D2H of the results, and returns
 * without synchronising; etx_wait_host(ticket) blocks until that submission has completed and returns its status
 * (ETX_ERR_INPUT_ORDER for a rejected batch).  At most TWO submissions may be in flight per handle: wait for
 * submission i before submitting i + 2, and give the two in-flight submissions different output buffers.  All output
 * buffers must be pinned (page-locked) host memory.  The edge list and the scores of submission i are copied out, at
 * their exact size, by the next call on the handle -- the submission of i + 1 or the wait for i -- once the host has
 * learnt E, which S3 produced long before: the edge list under batch i's own GNN, the scores under batch i + 1 (each
 * slot has its own device score buffer).  *h_n_edges (plain host int32) receives E and is valid after etx_wait_host.
 * While a submission has not been waited for, etx_run / etx_run_host / etx_dbg_run on the same handle return
 * ETX_ERR_ARG (they would overwrite its results).  The h_* input arrays and
 * h_event_offsets must stay valid until the submission has completed (h_event_offsets: until the call returns).
 * A submission slot is released by etx_wait_host only: submitting i + 2 before waiting for i returns ETX_ERR_ARG and
 * leaves the two submissions in flight untouched.  The first etx_submit_host on a handle allocates a second input
 * staging set and score buffer through the handle's allocator (etx_workspace_bytes grows by 16 max_hits + 4 k max_hits
 * bytes); a first call that fails half-way is completed by the next one. */
etx_status etx_submit_host(etx_handle h, const float* h_xyz, const int32_t* h_plane,
                           const int32_t* h_event_offsets, int32_t n_events, etx_stream stream,
                           float* h_edge_score, int32_t* h_edge_src, int32_t* h_edge_dst,
                           int32_t* h_track_id, int32_t* h_n_edges, int32_t* ticket);
etx_status etx_wait_host(etx_handle h, int32_t ticket);

/* Verdict of the device-side input validation for the last etx_run / etx_dbg_run on this handle whose stream work
 * has completed (the caller synchronises the stream first): ETX_OK, or ETX_ERR_INPUT_ORDER if that batch was
 * rejected.  Always ETX_OK when validate_input = 0. */
etx_status etx_input_status(etx_handle h);

/* Track containers (L42: a particle is reconstructible with at least three VELO hits; L74, L82: the product of
 * the pipeline is the set of tracks, each a list of hits).  Enqueue on `stream`, after an etx_run on the same
 * stream and handle, the regrouping of its track ids: a track is a component with at least min_hits hits; tracks
 * are numbered densely in ascending order of their smallest hit index (so the tracks of an event are
 * consecutive); the hits of a track are listed in ascending hit index.  Library-owned device pointers, valid
 * until the next call on the handle; no synchronisation. */
typedef struct {
  const int32_t* d_track_index;          /* [n_hits]        dense track number of the hit, or -1            */
  const int32_t* d_track_offsets;        /* [n_tracks + 1]  CSR offsets into d_track_hits                   */
  const int32_t* d_track_hits;           /* [offsets[n_tracks]] hit indices, track after track              */
  const int32_t* d_event_track_offsets;  /* [n_events + 1]  first track number of every event               */
  const int32_t* d_n_tracks;             /* device scalar                                                   */
  const int32_t* h_n_tracks;             /* pinned host mirror; valid once the stream has been synchronised */
} etx_tracks_output;

etx_status etx_tracks(etx_handle h, int32_t min_hits, etx_stream stream, etx_tracks_output* out);

/* The same regrouping for callers that are not allowed to allocate device memory: no handle, no workspace, and the
 * call itself never calls cudaMalloc / cudaFree or any routine that allocates -- it only enqueues kernels and
 * cudaMemsetAsync on `stream`.  It is meant for code that runs inside a host framework which owns all device memory and
 * forbids allocation in its event loop (Allen, hands every algorithm slices of a per-stream arena
 * sized in advance: cudaMalloc / cudaFree there would take the device-wide allocator lock and can stall the other
 * streams of events), and for plug-ins that are given raw device pointers and nothing else.
 *   inputs  (device, borrowed)  d_track_id [n_hits]         as etx_output.d_track_id: the smallest hit index of the
 *                                                           hit's component (values in [0, n_hits), track_id[r] == r
 *                                                           for that smallest hit, a component inside one event)
 *                               d_event_offsets [n_events+1] [0] = 0, non-decreasing, [n_events] = n_hits -- on the
 *                                                           DEVICE here (etx_run takes them from the host)
 *   outputs (device, caller's)  d_track_index [n_hits], d_track_offsets [n_hits + 1] (entries [0 .. n_tracks] are the
 *                               CSR offsets, later entries repeat the total), d_track_hits [n_hits] (the first
 *                               offsets[n_tracks] entries are written), d_event_track_offsets [n_events + 1],
 *                               d_n_tracks [1].  Same meaning and same values as etx_tracks_output.
 * Its work arrays live in a fixed array inside the library image instead: about 16 MiB of device memory on every GPU
 * that loads libetx.so, held until the process exits.  What follows from that:
 *   - n_hits > ETX_TRACKS_STATIC_MAX_HITS returns ETX_ERR_CAPACITY and launches nothing (split the batch at an event
 *     boundary, or use etx_tracks).  n_events is not limited.
 *   - The first call on each device resolves the array's device address (cudaGetSymbolAddress, once per device, with
 *     that device current, return code checked).  Make that first call before any stream capture is begun.
 *   - Every call on a GPU uses the same array and finds the previous call's contents in it; the call zeroes what it
 *     needs zeroed.  Calls whose device work can overlap on one GPU (two streams, two threads) race on it: keep them on
 *     one stream or order them with events.  Calls on different GPUs are independent.
 * No synchronisation; results are valid once `stream` has reached the end of the enqueued work.  Returns ETX_ERR_ARG
 * for null pointers, negative sizes or min_hits < 1, ETX_ERR_CUDA if a launch fails; etx_tracks_static_error() gives
 * the message of the last failing call on the calling thread ("" if the last call succeeded). */
#define ETX_TRACKS_STATIC_MAX_HITS (1 << 20)
etx_status etx_tracks_static(const int32_t* d_track_id, const int32_t* d_event_offsets, int32_t n_hits,
                             int32_t n_events, int32_t min_hits, etx_stream stream, int32_t* d_track_index,
                             int32_t* d_track_offsets, int32_t* d_track_hits, int32_t* d_event_track_offsets,
                             int32_t* d_n_tracks);
const char* etx_tracks_static_error(void);

/* Triplet stage (sec. 5.3; R28, R29), the step the paper left out of its CUDA code
 * (L238).  Enqueue on `stream`, after an etx_run on the same stream and handle: triplet building on the purified
 * hit graph (edges with logit >= tau) and the two triplet classifiers on pairs of final edge encodings.  Needs a
 * blob that carries the triplet classifiers (header word 11) and max_triplets > 0.  For kind k (0 articulation
 * A->C, C->B: first = the in-edge of the common hit C, second = its out-edge; 1 left elbow C->A, C->B; 2 right elbow
 * A->C, B->C; first < second for the elbows) the triplets are listed in ascending (C, first, second) order:
 *   d_first[k], d_second[k]  [count[k]] edge ids      d_hit[k]  [count[k]] the common hit
 *   d_logit[k], d_score[k]   [count[k]] classifier output (articulation classifier for kind 0, elbow classifier else)
 * d_count / h_count [3]: the number of triplets of each kind (h_count: pinned mirror, valid after synchronising).  If
 * a count exceeds max_triplets only the first max_triplets triplets of that kind are listed (the caller compares).
 * Counts are int32 and saturate: 2^31 - 1 means "at least 2^31 - 1" (they never wrap to a negative number).
 * Library-owned device pointers, valid until the next call on the handle; no synchronisation. */
typedef struct {
  const int32_t* d_first[3];
  const int32_t* d_second[3];
  const int32_t* d_hit[3];
  const float*   d_logit[3];
  const float*   d_score[3];
  const int32_t* d_count;
  const int32_t* h_count;
  int32_t        capacity;
} etx_triplets_output;

etx_status etx_triplets(etx_handle h, etx_stream stream, etx_triplets_output* out);

/* Track building from triplets, phases (1)-(2) (sec. 5.4; R30).  Enqueue after
 * etx_triplets on the same stream and handle.  Triplets are kept iff logit >= tau_t (triplet_threshold).  The two
 * edges of every kept elbow are merged into a super-edge; kept articulations are mapped onto super-edges (duplicates
 * collapse); an articulation is SHARED iff its first super-edge has >= 2 distinct successors or its second >= 2
 * distinct predecessors; the other articulations connect their super-edges.  Results:
 *   d_edge_component [n_edges]  for a kept edge the name of its set of connected edges = the smallest edge id in it,
 *                               -1 for an edge below the edge threshold
 *   d_shared [n_shared][2]      the shared articulations as (component of first, component of second); unordered and
 *                               possibly repeated -- a set (each yields the track "union of the two components",
 *                               phase 3; etx_triplet_tracks lists the tracks, phases 3-4)
 * Exact only if no triplet count exceeded max_triplets (compare etx_triplets' counts).  No synchronisation. */
typedef struct {
  const int32_t* d_edge_component;
  const int32_t* d_shared;
  const int32_t* d_n_shared;
  const int32_t* h_n_shared;             /* pinned mirror; valid once the stream has been synchronised */
  int32_t        capacity;               /* pairs d_shared can hold (= max_triplets)                    */
} etx_triplet_components_output;

etx_status etx_triplet_components(etx_handle h, etx_stream stream, etx_triplet_components_output* out);

/* Track building from triplets, phases (3)-(4) (sec. 5.4: "a new track is formed for each remaining
 * articulation, effectively duplicating the shared set of connected edges.  Finally, edges are replaced by their
 * corresponding hits"; Fig. 6; R30, R31).  Enqueue after etx_triplet_components on the same stream and
 * handle.  Every shared articulation (X, Y) gives the track "hits of set X and of set Y"; a set of connected edges that
 * no shared articulation touches is a track by itself; a track's hits are the end points of its edges.  Hits ascend
 * inside a track; tracks with fewer than min_hits hits are dropped (L42: 3); identical hit lists are kept once; tracks
 * are ordered lexicographically by hit list -- so tracks may share hits, which is the point of the triplet stage (e+e-
 * pairs, L166).  Results (library-owned device memory, valid until the next call on the handle; no synchronisation):
 *   d_track_offsets [n_tracks + 1]  CSR offsets into d_track_hits          d_track_hits [offsets[n_tracks]]
 *   d_counts / h_counts [3]         n_tracks, total number of listed hits, overflow flag (h_counts: pinned mirror,
 *                                   valid once the stream has been synchronised)
 * Capacities: track_capacity = max_triplets + k * max_hits tracks (never exceeded: at most one track per shared
 * articulation and per set) and hit_capacity = 2 * track_capacity listed hits (a shared set is listed once per
 * articulation that shares it, so there is no bound in terms of n_hits); if the latter is exceeded the
 * overflow flag is 1, the counts are the true ones and the lists are cut there.  Exact only if etx_triplets' counts
 * stayed within max_triplets.  Needs max_triplets + k * max_hits < 2^31 (ETX_ERR_UNSUPPORTED otherwise). */
typedef struct {
  const int32_t* d_track_offsets;
  const int32_t* d_track_hits;
  const int32_t* d_counts;
  const int32_t* h_counts;
  int32_t        track_capacity;
  int32_t        hit_capacity;
} etx_triplet_tracks_output;

etx_status etx_triplet_tracks(etx_handle h, int32_t min_hits, etx_stream stream, etx_triplet_tracks_output* out);

/* INT8 calibration (sec. 7.4: the quantised model is "calibrated" on a sample of events; DESIGN.md
 * R21): the activation scales an INT8 blob needs, one per quantised Linear (K >= 16, not the d -> 1
 * heads) in blob order.  Runs the whole fp32 path S0..S5 (and, if the blob carries triplet classifiers, the triplet
 * stage) over the given calibration batch on a handle created with precision ETX_FP32, keeps on the device the running
 * max |x| of every such Linear's input tensor (rows that exist only; max is order-free, so the result is reproducible),
 * and returns s_x = max|x| / 127 (true fp32 division; 1.0 if the maximum is 0) in h_scales [*n_scales].  The blob of
 * the INT8 handle is then the same weights followed by these scales (datagen/weights.py: header word 9 = their count).
 *   d_xyz, d_plane, h_event_offsets, n_events   a batch, as for etx_run
 *   h_scales [capacity]  host, written on ETX_OK; NULL: only *n_scales (the count the model needs) is returned
 * Synchronises `stream`.  ETX_ERR_UNSUPPORTED on a handle that is not ETX_FP32; ETX_ERR_CAPACITY if capacity is too
 * small, or if the blob has triplet classifiers and max_triplets is 0 or was exceeded by the batch.  The first call
 * allocates one small device array through the handle's allocator. */
etx_status etx_calibrate(etx_handle h, const float* d_xyz, const int32_t* d_plane, const int32_t* h_event_offsets,
                         int32_t n_events, etx_stream stream, float* h_scales, int32_t capacity, int32_t* n_scales);

etx_status etx_destroy(etx_handle h);

/* Device bytes held by the handle (workspace + converted weights), as requested from the allocator. */
size_t etx_workspace_bytes(etx_handle h);

const char* etx_status_string(etx_status s);
const char* etx_last_error(etx_handle h);         /* message of the last failing call on this handle */

/* ---------------------------------------------------------------------------
 * Debug / measurement entry points (not part of the three-call contract).  They exist for the
 * stage-isolated parity protocol: a stage is bit-exact only for identical inputs
 * to that stage, so the tests inject the oracle's embedding / edge list / logits.
 * -------------------------------------------------------------------------*/
typedef struct {
  const float*   d_emb;        /* non-NULL: skip S1 and use this [n_hits][emb_dim] embedding           */
  const int32_t* d_src;        /* non-NULL (with d_dst): skip S2 + pack and use this edge list; it must */
  const int32_t* d_dst;        /*   be sorted by src; row_ptr / CSC are rebuilt from it                 */
  int32_t        n_edges;
  const float*   d_logit;      /* non-NULL: skip S4 and use these [n_edges] logits                      */
  int32_t        last_stage;   /* stop after stage 1..5 (5 = run everything)                            */
} etx_inject;

etx_status etx_dbg_run(etx_handle h, const float* d_xyz, const int32_t* d_plane,
                       const int32_t* h_event_offsets, int32_t n_events, etx_stream stream,
                       const etx_inject* inj, etx_output* out);

/* Device pointer + byte size of an internal buffer of the last run: "plane_off", "emb", "nbr", "deg",
 * "row_ptr", "col_ptr", "in_edge", "h", "e", "m", "logit", "tap", "feat", "feat_emb", "trip_logit" ([3][max_triplets]
 * classifier outputs of etx_triplets; the fixture tests overwrite them to choose which triplets are kept).  "nbr" is [n_hits][k]; only the
 * first deg[q] slots of a row are defined.  h / e / m are in the
 * state dtype (etx_state_dtype; by default fp32 for ETX_FP32 and ETX_INT8, bf16 for ETX_BF16).  "e" holds the final edge state e^L only after
 * etx_dbg_run: in etx_run the last edge network feeds the fused classifier and does not write e^L back (the
 * tensor-core kernels; after etx_run "e" is then e^(L-1)). */
etx_status etx_dbg_buffer(etx_handle h, const char* name, const void** d_ptr, size_t* bytes);

/* INT8 only: record the int32 accumulators of Linear `layer_index` (blob order) of the next run into
 * the "tap" buffer ([rows][out] int32); -1 switches it off. */
etx_status etx_dbg_tap_layer(etx_handle h, int32_t layer_index);

/* Per-stage device times of the last etx_run / etx_dbg_run in milliseconds (CUDA events recorded on
 * the run's stream; valid after the stream is synchronised).  Order: S0, S1, S2, S3, S4 encoders,
 * S4 scatter (sum over steps), S4 node nets, S4 edge nets (+ head), S5.  Recording is enabled by
 * etx_dbg_enable_timing(h, 1). */
#define ETX_N_STAGE_TIMES 9
etx_status etx_dbg_enable_timing(etx_handle h, int32_t on);
etx_status etx_dbg_stage_times(etx_handle h, float* ms_out /* [ETX_N_STAGE_TIMES] */);

/* Number of kernels this library launched since the handle was created (bench.py's gpu_launches). */
int64_t etx_dbg_launch_count(etx_handle h);

#ifdef __cplusplus
}
#endif
#endif  /* ETX_H_ */
