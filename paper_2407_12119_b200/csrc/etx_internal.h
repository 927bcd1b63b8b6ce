// Internal declarations of the ETX4VELO B200 library (not part of the C-ABI; see include/etx.h).
// Shares nothing with oracle/ (the CPU oracle is test infrastructure and has its own code).
#pragma once

#include <cuda_bf16.h>
#include <cuda_runtime.h>
#include <stdint.h>

#include <string>
#include <utility>
#include <vector>

#include "../../include/etx.h"

namespace etx {

constexpr int kMaxEmbLayers = 9;     // H + 1, H <= 8
constexpr int kTileRows = 64;        // rows (hits / edges) per CTA tile of the FFMA embedding / triplet kernels
constexpr int kGnnRows = 128;        // rows per CTA tile of the FFMA interaction-network kernels
constexpr int kGnnThreads = 512;     // ... and their threads (one CTA per SM at d = 64: 16 warps hide the FFMA / LDS latencies)
constexpr int kMlpThreads = 256;

// One Linear, as the kernels see it.  W is stored transposed ([K][N], N contiguous) in fp32 holding the
// values the precision mode multiplies with: the fp32 weights, their bf16 roundings, or the int8 codes.
struct LayerP {
  const float* Wt;        // [K][N]
  const float* scale;     // [N]  y = fmaf(acc, scale, bias); 1.0 except INT8 tensor layers (s_x * s_w[c])
  const float* bias;      // [N]
  const void* Wtc;        // tensor-core operand: W[N][K] K-major, bf16 or int8, swizzled per K-block
  float inv_sx;           // INT8 tensor layers: 1 / s_x of the layer's input tensor
  int K, N;
  int tensor;             // K >= 16 and not the head (R20 / R21)
  int index;              // position in blob order
};

enum MlpKind { kNodeEnc = 0, kEdgeEnc = 1, kNodeNet = 2, kEdgeNet = 3 };

struct GnnArgs {
  LayerP l0, l1, head;
  const float4* feat;        // [n_hits] normalised (fx, fy, fz, 0)
  const int32_t* src;        // [E]
  const int32_t* dst;        // [E]
  const int32_t* n_rows_ptr; // device scalar: number of rows (E for edge kernels), or nullptr -> n_rows
  int n_rows;
  void* h;                   // [n_hits][d]  state dtype
  void* e;                   // [E][d]
  const void* m;             // [n_hits][2d]
  float* logit;              // [E]  (do_head)
  float* score;              // [E]
  int do_head;
  int edge_enc_input;
  int32_t* tap;              // int32 accumulators of layer tap_layer, or nullptr
  int tap_layer;
  // INT8, warp-specialised kernels: the node network also stores the int8 codes of the new h under the NEXT edge
  // network's input scale (hq_out, hq_inv_sx); the edge network gathers those codes (hq_in) instead of re-quantising
  // h[src] / h[dst] for every edge.  nullptr: quantise on the fly.
  int8_t* hq_out = nullptr;
  float hq_inv_sx = 1.0f;
  const int8_t* hq_in = nullptr;
  float* absmax = nullptr;   // etx_calibrate (FFMA kernels, fp32 mode): running max |x| per layer in blob order, or nullptr
};

struct EmbArgs {
  LayerP layers[kMaxEmbLayers];
  int n_layers;              // H + 1
  const float4* feat;
  float4* emb;               // [n_hits] (emb_dim == 4)
  int n_rows;
  int32_t* tap;
  int tap_layer;
  float* absmax = nullptr;    // etx_calibrate: running max |x| per layer (blob order), or nullptr
};

struct HostLayer {
  int out = 0, in = 0, index = 0;
  bool tensor = false;
  std::vector<float> W, b;       // blob values
  float sx = 1.0f;
  LayerP dev{};
};

}  // namespace etx

struct etx_ctx {
  etx_hyperparams hp{};
  int precision = 0, engine = 0;
  bool state_bf16 = false;
  int max_edges = 0;
  int sm_count = 148;
  int device = 0;                         // the CUDA device the handle was created on (tensor maps, sm_count, opt-ins)
  std::vector<std::pair<const void*, int>> smem_opted;   // kernels whose dynamic shared-memory limit was raised for this handle
  std::string error;
  std::vector<etx::HostLayer> layers;     // blob order
  int i_emb0 = 0, i_nenc = 0, i_eenc = 0, i_iter0 = 0, i_head = 0, i_trip = -1;   // i_trip: the four triplet-classifier layers, or -1
  std::vector<void*> allocs;              // every device block of this handle (etx_device_alloc)
  size_t device_bytes = 0;
  // workspace
  int32_t* event_off = nullptr;           // [max_events + 1]
  int32_t* plane_off = nullptr;           // [max_events][P + 1]
  float4* feat = nullptr;                 // [max_hits]
  bool keep_final_state = false;          // etx_dbg_run: the last edge network still writes e^L (tests read it)
  int32_t* knn_redo = nullptr;            // [max_events * n_planes] buckets knn_cut_kernel hands to knn_kernel
  float4* feat_emb = nullptr;             // [max_hits] input of the embedding MLP (= feat unless emb_input = 1)
  float4* emb = nullptr;                  // [max_hits]
  int32_t *nbr = nullptr, *deg = nullptr; // [max_hits][k], [max_hits]
  int32_t *row_ptr = nullptr, *col_ptr = nullptr, *cursor = nullptr;   // [max_hits + 1]
  int32_t *src = nullptr, *dst = nullptr, *in_edge = nullptr;          // [max_edges]
  int32_t* scan_tmp = nullptr;            // block sums
  int32_t* n_edges = nullptr;             // device scalar
  int32_t* flags = nullptr;               // device: [0] input-order violation
  void *h = nullptr, *e = nullptr, *m = nullptr;
  float *logit = nullptr, *score = nullptr;
  float* score_out = nullptr;             // where the classifier writes scores: `score`, or the caller's mapped host buffer (etx_run_host)
  int32_t *track_id = nullptr;
  // track containers (etx_tracks): component sizes, keep flags / cursors, dense numbers, kept sizes, outputs
  int32_t *trk_size = nullptr, *trk_keep = nullptr, *trk_number = nullptr, *trk_ksize = nullptr;
  int32_t *trk_index = nullptr, *trk_offsets = nullptr, *trk_hits = nullptr, *trk_event_off = nullptr;
  int32_t *n_tracks = nullptr, *h_n_tracks = nullptr;
  // triplet stage (etx_triplets): per-hit counts / offsets [3][max_hits + 1], triplets [3][max_triplets]
  int32_t *trip_cnt = nullptr, *trip_off = nullptr, *trip_first = nullptr, *trip_second = nullptr, *trip_hit = nullptr;
  float *trip_logit = nullptr, *trip_score = nullptr;
  int32_t *trip_total = nullptr, *h_trip_total = nullptr;   // [3] device / pinned
  // etx_triplet_components: union-find parents over edges (elbows; non-shared articulations), distinct successor /
  // predecessor counts, hash set of (super-edge, super-edge) pairs, outputs
  int32_t *tc_par1 = nullptr, *tc_par2 = nullptr, *tc_succ = nullptr, *tc_pred = nullptr, *tc_comp = nullptr, *tc_shared = nullptr;
  unsigned long long* tc_tab = nullptr;
  size_t tc_tab_size = 0;
  int32_t *tc_n_shared = nullptr, *h_tc_n_shared = nullptr;
  float tau_t = 0.0f;
  // etx_triplet_tracks (k_triplet_tracks.cu): hit lists of the sets of connected edges (CSR by set name), candidate
  // numbers bucketed by first hit, the track list, {n_tracks, total hits, overflow} device / pinned
  int32_t *tt_set_off = nullptr, *tt_set_hits = nullptr, *tt_bucket_cand = nullptr, *tt_scan_tmp = nullptr;
  int32_t *tt_track_len = nullptr, *tt_track_off = nullptr, *tt_track_hits = nullptr, *tt_counts = nullptr, *h_tt_counts = nullptr;
  int tt_hit_cap = 0, tt_track_cap = 0;
  int last_n_events = 0;
  // k_edge_tma.cu: identity operand image, split-bias images [2 * iter + layer], CUtensorMap of `e` (opaque here)
  bool edge_tma = false;
  bool edge_i8 = false;                   // k_edge_i8.cu usable (INT8, auto engine, tensor map of fp32 `e` encoded)
  void* ident_img = nullptr;
  void* eenc_b0_img = nullptr;
  void* eenc_b1_img = nullptr;
  void* nenc_b1_img = nullptr;
  void* trip_b0_img[2] = {nullptr, nullptr};   // split-bias images of the two triplet classifiers' first layer
  void* zero_bias_img = nullptr;
  std::vector<void*> edge_bias_img;
  alignas(64) unsigned char e_map[128] = {};
  alignas(64) unsigned char h_map[128] = {};   // CUtensorMap of `h` (node encoder output)
  int8_t* hq = nullptr;                   // [max_hits][d] int8 codes of h for the edge network (INT8, AUTO engine)
  int32_t* tap = nullptr;
  size_t tap_bytes = 0;
  int tap_layer = -1;
  float* absmax = nullptr;                // [layers] etx_calibrate: max |x| of every Linear's input (device)
  bool calibrating = false;
  // host side
  int32_t* h_event_off = nullptr;         // pinned staging [max_events + 1]
  int32_t* h_n_edges = nullptr;           // pinned mirror
  int32_t* h_flags = nullptr;             // pinned mirror
  cudaEvent_t staging_free = nullptr;
  cudaEvent_t edges_ready = nullptr, copies_done = nullptr;   // etx_run_host: src / dst D2H under the GNN
  cudaStream_t copy_stream = nullptr;
  // staging for etx_run_host
  float* d_xyz_in = nullptr;
  int32_t* d_plane_in = nullptr;
  // etx_submit_host / etx_wait_host: a second input staging set, one completion event, "inputs consumed" event and
  // validation flag per slot (two submissions may be in flight)
  float* d_xyz_in2 = nullptr;
  int32_t* d_plane_in2 = nullptr;
  cudaEvent_t slot_done[2] = {nullptr, nullptr}, slot_inputs_read[2] = {nullptr, nullptr}, slot_h2d[2] = {nullptr, nullptr};
  int32_t* h_slot_flags = nullptr;        // pinned [2]
  int32_t* h_flags_cur = nullptr;         // where run_impl mirrors the validation flag of the batch it enqueues
  cudaEvent_t inputs_read_cur = nullptr;  // recorded by run_impl once S0 has read xyz / plane (or nullptr)
  cudaEvent_t edges_ready_cur = nullptr;  // run_impl records this instead of edges_ready when set
  int32_t* h_n_edges_cur = nullptr;       // ... and mirrors E here instead of h_n_edges
  cudaEvent_t slot_edges_ready[2] = {nullptr, nullptr}, slot_copies_done[2] = {nullptr, nullptr};
  int32_t* h_slot_n_edges = nullptr;      // pinned [2]
  struct PendingCopy { int32_t* h_src = nullptr; int32_t* h_dst = nullptr; int32_t* h_n = nullptr; float* h_score = nullptr;
                       const float* d_score = nullptr; bool pending = false; } slot_copy[2];
  cudaEvent_t slot_edges_copied[2] = {nullptr, nullptr};
  float* score2 = nullptr;                // second score buffer: the scores of submission i are copied out under batch i + 1
  cudaStream_t h2d_stream = nullptr;      // inputs of the next submission (PCIe is full duplex: D2H runs on copy_stream)
  long long n_submitted = 0;
  bool slot_unwaited[2] = {false, false}; // set by etx_submit_host, cleared by etx_wait_host only (not by the edge-list flush)
  bool submit_ready = false;              // the lazily created submit resources all exist
  // timing
  bool timing = false;
  cudaEvent_t ev[256] = {};
  int n_ev = 0;
  struct Span { int a, b, stage; };
  std::vector<Span> spans;
  int64_t launches = 0;
  int last_n_hits = 0;
  float tau = 0.0f;
};

namespace etx {

// cudaFuncAttributeMaxDynamicSharedMemorySize is a per-DEVICE setting, so the opt-in is remembered per handle (a handle
// lives on one device), not per process; a larger request for the same kernel raises the limit again.
template <typename K>
inline void opt_in_smem(etx_ctx* c, K kern, int bytes) {
  const void* f = reinterpret_cast<const void*>(kern);
  for (auto& e : c->smem_opted)
    if (e.first == f) {
      if (e.second >= bytes) return;
      cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, bytes);
      e.second = bytes;
      return;
    }
  cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, bytes);
  c->smem_opted.push_back({f, bytes});
}

// ---- launchers (each file owns its kernels) -------------------------------------------------------------
// etx_api.cu: device memory through the handle's allocator (hp.alloc or cudaMalloc); nullptr on failure
void* etx_device_alloc(etx_ctx* c, size_t bytes);
// k_graph.cu
void launch_features(etx_ctx* c, const float* xyz, int n_hits, cudaStream_t s);
void launch_edge_enc_h_tma(etx_ctx* c, int n_hits, bool do_head, cudaStream_t s);
void launch_plane_offsets(etx_ctx* c, const int32_t* plane, int n_events, cudaStream_t s);
void launch_validate(etx_ctx* c, const int32_t* plane, int n_events, int n_hits, cudaStream_t s);
void launch_knn(etx_ctx* c, const int32_t* plane, int n_events, int n_hits, cudaStream_t s);
void launch_pack_edges(etx_ctx* c, int n_hits, cudaStream_t s);                 // deg, nbr -> row_ptr, src, dst, n_edges
void launch_rows_from_src(etx_ctx* c, int n_hits, int n_edges, cudaStream_t s); // injected edge list -> row_ptr
void launch_csc(etx_ctx* c, int n_events, int n_hits, bool windowed, cudaStream_t s);                        // dst -> col_ptr, in_edge
void launch_components(etx_ctx* c, const float* logit, int n_events, int n_hits, cudaStream_t s);
void launch_tracks(etx_ctx* c, int n_events, int n_hits, int min_hits, cudaStream_t s);
void launch_triplet_build(etx_ctx* c, int n_hits, cudaStream_t s);
void launch_triplet_components(etx_ctx* c, cudaStream_t s);
// k_triplet_tracks.cu
void launch_triplet_tracks(etx_ctx* c, int n_events, int n_hits, int min_hits, cudaStream_t s);
// k_mlp_simt.cu
void launch_embed_simt(etx_ctx* c, int n_hits, cudaStream_t s);
void launch_gnn_mlp_simt(etx_ctx* c, int kind, int iter, int n_hits, bool do_head, cudaStream_t s);
void launch_scatter(etx_ctx* c, int n_hits, cudaStream_t s);
void simt_configure(etx_ctx* c);
void launch_triplet_classifier(etx_ctx* c, int kind, cudaStream_t s);
void fill_gnn_args(etx_ctx* c, int kind, int iter, int n_hits, bool do_head, GnnArgs& a);
// k_mlp_umma.cu
bool umma_supported(const etx_ctx* c);
void umma_configure(etx_ctx* c);
void launch_embed_umma(etx_ctx* c, int n_hits, cudaStream_t s);
void launch_gnn_mlp_umma(etx_ctx* c, int kind, int iter, int n_hits, bool do_head, cudaStream_t s);
// k_mlp_ws.cu (bf16: warp-specialised, pipelined)
void launch_gnn_mlp_ws(etx_ctx* c, int kind, int iter, int n_hits, bool do_head, cudaStream_t s);

// k_edge_i8.cu (int8: warp-specialised edge network with quantising producers)
bool edge_i8_configure(etx_ctx* c);
void launch_edge_net_i8(etx_ctx* c, int iter, int n_hits, bool do_head, cudaStream_t s);
void launch_node_net_i8(etx_ctx* c, int iter, int n_hits, cudaStream_t s);
// k_embed_ws.cu (bf16: four tiles in flight per SM; false = shape not covered, nothing launched)
bool launch_embed_ws(etx_ctx* c, int n_hits, cudaStream_t s);
// k_edge_tma.cu (bf16: the edge network with TMA-moved edge state, bias and residual inside the MMAs)
bool edge_tma_configure(etx_ctx* c);
void launch_edge_net_tma(etx_ctx* c, int iter, int n_hits, bool do_head, cudaStream_t s);
void launch_edge_enc_tma(etx_ctx* c, int n_hits, bool node, cudaStream_t s);
void launch_triplet_cls_tma(etx_ctx* c, int kind, cudaStream_t s);

}  // namespace etx
