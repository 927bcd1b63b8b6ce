// C-ABI entry points (include/etx.h): blob parsing, weight conversion, workspace, the stream-ordered launch
// sequence S0..S5.  No host synchronisation inside etx_run; E lives on the device (n_edges) and every
// E-sized kernel reads it there.
#include <math.h>
#include <string.h>

#include <new>

#include <algorithm>

#include "etx_internal.h"

using namespace etx;

namespace {

constexpr uint32_t kBlobMagic = 0x57585445u;   // 'ETXW'

struct CudaFail { cudaError_t err; const char* what; };

#define ETX_CUDA(call)                                                                  \
  do {                                                                                  \
    cudaError_t err__ = (call);                                                         \
    if (err__ != cudaSuccess) throw CudaFail{err__, #call};                             \
  } while (0)

template <typename T>
T* dev_alloc(etx_ctx* c, size_t n) {
  void* p = etx::etx_device_alloc(c, (n ? n : 1) * sizeof(T));
  if (!p) throw CudaFail{cudaErrorMemoryAllocation, "device allocation"};
  return static_cast<T*>(p);
}

float* upload(etx_ctx* c, const std::vector<float>& v) {
  float* p = dev_alloc<float>(c, v.size());
  ETX_CUDA(cudaMemcpy(p, v.data(), v.size() * sizeof(float), cudaMemcpyHostToDevice));
  return p;
}

float host_bf16_round(float x) { return __bfloat162float(__float2bfloat16_rn(x)); }

etx_status fail(etx_ctx* c, etx_status st, const std::string& msg) {
  if (c) c->error = msg;
  return st;
}

// Blob layout: datagen/weights.py header comment (and include/etx.h, etx_create).
etx_status parse_blob(etx_ctx* c, const uint8_t* blob, size_t bytes) {
  const etx_hyperparams& hp = c->hp;
  if (bytes < 64) return fail(c, ETX_ERR_BLOB, "blob smaller than its header");
  uint32_t h[16];
  memcpy(h, blob, 64);
  if (h[0] != kBlobMagic || h[1] != 1u) return fail(c, ETX_ERR_BLOB, "bad blob magic / version");
  if ((int)h[2] != hp.emb_hidden || (int)h[3] != hp.emb_n_hidden_layers || (int)h[4] != hp.emb_dim ||
      (int)h[5] != hp.gnn_latent || (int)h[6] != hp.gnn_iters || (int)h[7] != hp.edge_enc_input || (int)h[10] != hp.emb_input)
    return fail(c, ETX_ERR_BLOB, "blob shapes differ from the hyper-parameters");
  const int D = hp.emb_hidden, H = hp.emb_n_hidden_layers, d = hp.gnn_latent, L = hp.gnn_iters;
  auto add = [&](int out, int in, bool head = false) {
    HostLayer l;
    l.out = out; l.in = in; l.index = (int)c->layers.size();
    l.tensor = (in >= 16) && !head;
    c->layers.push_back(l);
  };
  c->i_emb0 = 0;
  add(D, 3);
  for (int i = 1; i < H; ++i) add(D, D);
  add(hp.emb_dim, D);
  c->i_nenc = (int)c->layers.size();
  add(d, 3); add(d, d);
  c->i_eenc = (int)c->layers.size();
  add(d, hp.edge_enc_input ? 2 * d : 3); add(d, d);
  c->i_iter0 = (int)c->layers.size();
  for (int it = 0; it < L; ++it) { add(d, 3 * d); add(d, d); add(d, 3 * d); add(d, d); }
  c->i_head = (int)c->layers.size();
  add(1, d, true);
  if (h[11] > 1u) return fail(c, ETX_ERR_BLOB, "bad triplet-classifier flag");
  if (h[11] == 1u) {                 // L160: articulation classifier, elbow classifier: 2d -> d -> 1 (R28)
    c->i_trip = (int)c->layers.size();
    add(d, 2 * d); add(1, d, true);
    add(d, 2 * d); add(1, d, true);
  }
  size_t need = 0; int nq = 0;
  for (auto& l : c->layers) { need += (size_t)l.out * l.in + l.out; nq += l.tensor; }
  if (h[8] != need) return fail(c, ETX_ERR_BLOB, "blob weight count differs from the shapes");
  const size_t n_scales = h[9];
  if (bytes != 64 + 4 * (need + n_scales)) return fail(c, ETX_ERR_BLOB, "blob size mismatch");
  if (c->precision == ETX_INT8 && (int)n_scales != nq)
    return fail(c, ETX_ERR_BLOB, "INT8 needs one activation scale per Linear with K >= 16");
  const float* p = reinterpret_cast<const float*>(blob + 64);
  const float* scales = p + need;
  int qi = 0;
  for (auto& l : c->layers) {
    l.W.assign(p, p + (size_t)l.out * l.in); p += (size_t)l.out * l.in;
    l.b.assign(p, p + l.out); p += l.out;
    if (c->precision == ETX_INT8 && l.tensor) {
      l.sx = scales[qi++];
      if (!(l.sx > 0.0f) || !isfinite(l.sx)) return fail(c, ETX_ERR_BLOB, "activation scale must be finite and > 0");
    }
  }
  return ETX_OK;
}

// fp32 -> the operand set of the precision mode (R20 bf16 RNE; R21 symmetric per-channel int8)
void convert_layer(etx_ctx* c, HostLayer& l) {
  const int K = l.in, N = l.out;
  std::vector<float> Wt((size_t)K * N), scale(N, 1.0f);
  std::vector<float> Wop((size_t)N * K);               // operand values, [N][K]
  float inv_sx = 1.0f;
  if (c->precision == ETX_INT8 && l.tensor) {
    inv_sx = 1.0f / l.sx;
    for (int n = 0; n < N; ++n) {
      float m = 0.0f;
      for (int k = 0; k < K; ++k) m = fmaxf(m, fabsf(l.W[(size_t)n * K + k]));
      const float sw = m > 0.0f ? m / 127.0f : 1.0f;
      scale[n] = l.sx * sw;
      for (int k = 0; k < K; ++k) {
        float r = nearbyintf(l.W[(size_t)n * K + k] / sw);
        r = fminf(127.0f, fmaxf(-127.0f, r));
        Wop[(size_t)n * K + k] = r;
      }
    }
  } else if (c->precision == ETX_BF16 && l.tensor) {
    for (size_t i = 0; i < Wop.size(); ++i) Wop[i] = host_bf16_round(l.W[i]);
  } else {
    Wop = l.W;
  }
  for (int n = 0; n < N; ++n)
    for (int k = 0; k < K; ++k) Wt[(size_t)k * N + n] = Wop[(size_t)n * K + k];
  l.dev.Wt = upload(c, Wt);
  l.dev.scale = upload(c, scale);
  l.dev.bias = upload(c, l.b);
  l.dev.Wtc = nullptr;
  l.dev.inv_sx = inv_sx;
  l.dev.K = K; l.dev.N = N; l.dev.tensor = l.tensor ? 1 : 0; l.dev.index = l.index;
  l.W.swap(Wop);   // keep the operand values for the tensor-core packer (umma_configure)
}

__global__ void set_scalar_kernel(int32_t* p, int32_t v) { *p = v; }
__global__ void sigmoid_kernel(const float* __restrict__ z, const int32_t* __restrict__ n, float* __restrict__ s) {
  const int E = *n;
  for (int i = blockIdx.x * blockDim.x + threadIdx.x; i < E; i += gridDim.x * blockDim.x) s[i] = 1.0f / (1.0f + expf(-z[i]));
}

struct StageTimer {
  etx_ctx* c; cudaStream_t s;
  void begin(int stage) {
    if (!c->timing || c->n_ev + 2 > 256) return;
    cudaEventRecord(c->ev[c->n_ev], s);
    c->spans.push_back({c->n_ev, -1, stage});
    c->n_ev++;
  }
  void end() {
    if (!c->timing || c->spans.empty() || c->spans.back().b >= 0 || c->n_ev + 1 > 256) return;
    cudaEventRecord(c->ev[c->n_ev], s);
    c->spans.back().b = c->n_ev++;
  }
};

etx_status run_impl(etx_ctx* c, const float* d_xyz, const int32_t* d_plane, const int32_t* h_eo, int n_events,
                    cudaStream_t s, const etx_inject* inj, etx_output* out) {
  if (!c) return ETX_ERR_ARG;
  if (!h_eo || n_events < 0 || !out) return fail(c, ETX_ERR_ARG, "null event offsets / output, or n_events < 0");
  if (n_events > c->hp.max_events) return fail(c, ETX_ERR_CAPACITY, "n_events exceeds max_events");
  if (h_eo[0] != 0) return fail(c, ETX_ERR_ARG, "event_offsets[0] must be 0");
  for (int e = 0; e < n_events; ++e)
    if (h_eo[e + 1] < h_eo[e]) return fail(c, ETX_ERR_ARG, "event_offsets must be non-decreasing");
  const int n_hits = h_eo[n_events];
  if (n_hits > c->hp.max_hits) return fail(c, ETX_ERR_CAPACITY, "n_hits exceeds max_hits");
  if (n_hits > 0 && (!d_xyz || !d_plane)) return fail(c, ETX_ERR_ARG, "null hit arrays");
  {
    int dev = -1;
    if (cudaGetDevice(&dev) != cudaSuccess || dev != c->device)
      return fail(c, ETX_ERR_ARG, "the current CUDA device is not the one the handle was created on");
  }
  const int last = inj ? (inj->last_stage > 0 ? inj->last_stage : 5) : 5;
  if (inj && ((inj->d_src == nullptr) != (inj->d_dst == nullptr))) return fail(c, ETX_ERR_ARG, "inject: src and dst go together");
  if (inj && inj->d_logit && !inj->d_src) return fail(c, ETX_ERR_ARG, "inject: logits need the edge list they belong to");
  if (inj && inj->d_src && (inj->n_edges < 0 || inj->n_edges > c->max_edges)) return fail(c, ETX_ERR_CAPACITY, "inject: n_edges exceeds k * max_hits");
  try {
    // event offsets: pinned staging -> device (the only H2D of the call)
    ETX_CUDA(cudaEventSynchronize(c->staging_free));
    memcpy(c->h_event_off, h_eo, sizeof(int32_t) * ((size_t)n_events + 1));
    ETX_CUDA(cudaMemcpyAsync(c->event_off, c->h_event_off, sizeof(int32_t) * ((size_t)n_events + 1), cudaMemcpyHostToDevice, s));
    ETX_CUDA(cudaEventRecord(c->staging_free, s));
    ETX_CUDA(cudaMemsetAsync(c->n_edges, 0, sizeof(int32_t), s));
    c->n_ev = 0; c->spans.clear();
    c->last_n_hits = n_hits; c->last_n_events = n_events;
    // e^L feeds only the classifier (L142), so a plain run does not write it back -- unless the triplet stage, which
    // reads pairs of final edge encodings (L80), can follow
    c->keep_final_state = (inj != nullptr) || (c->i_trip >= 0 && c->hp.max_triplets > 0);
    StageTimer tm{c, s};
    bool edges_marked = false;
    const bool tensor_engine = (c->precision != ETX_FP32) && c->engine != ETX_ENGINE_SIMT;
    if (n_hits > 0) {
      // ---- S0
      tm.begin(0);
      launch_features(c, d_xyz, n_hits, s);
      launch_plane_offsets(c, d_plane, n_events, s);
      if (c->hp.validate_input) launch_validate(c, d_plane, n_events, n_hits, s);
      if (c->inputs_read_cur) ETX_CUDA(cudaEventRecord(c->inputs_read_cur, s));   // S0 is the only reader of xyz / plane
      tm.end();
      // ---- S1
      tm.begin(1);
      if (inj && inj->d_emb) ETX_CUDA(cudaMemcpyAsync(c->emb, inj->d_emb, sizeof(float4) * (size_t)n_hits, cudaMemcpyDeviceToDevice, s));
      else if (tensor_engine) {
        if (!(c->engine == ETX_ENGINE_AUTO && launch_embed_ws(c, n_hits, s))) launch_embed_umma(c, n_hits, s);
      }
      else launch_embed_simt(c, n_hits, s);
      tm.end();
      if (last >= 2) {
        // ---- S2, S3
        if (inj && inj->d_src) {
          tm.begin(3);
          if (inj->n_edges > 0) {
            ETX_CUDA(cudaMemcpyAsync(c->src, inj->d_src, sizeof(int32_t) * (size_t)inj->n_edges, cudaMemcpyDeviceToDevice, s));
            ETX_CUDA(cudaMemcpyAsync(c->dst, inj->d_dst, sizeof(int32_t) * (size_t)inj->n_edges, cudaMemcpyDeviceToDevice, s));
          }
          set_scalar_kernel<<<1, 1, 0, s>>>(c->n_edges, inj->n_edges); c->launches++;
          launch_rows_from_src(c, n_hits, inj->n_edges, s);
        } else {
          tm.begin(2);
          launch_knn(c, d_plane, n_events, n_hits, s);
          tm.end();
          tm.begin(3);
          launch_pack_edges(c, n_hits, s);
        }
        // E and the edge list are final here: mirror E to the host and mark the point (etx_run_host starts the
        // D2H copy of src / dst on its copy stream from this event, under the GNN)
        ETX_CUDA(cudaMemcpyAsync(c->h_n_edges_cur ? c->h_n_edges_cur : c->h_n_edges, c->n_edges, sizeof(int32_t), cudaMemcpyDeviceToHost, s));
        ETX_CUDA(cudaEventRecord(c->edges_ready_cur ? c->edges_ready_cur : c->edges_ready, s));
        edges_marked = true;
        if (last >= 3) launch_csc(c, n_events, n_hits, !(inj && inj->d_src), s);
        tm.end();
      }
      if (last >= 4) {
        // ---- S4
        if (inj && inj->d_logit) {
          tm.begin(7);
          if (inj->n_edges > 0) ETX_CUDA(cudaMemcpyAsync(c->logit, inj->d_logit, sizeof(float) * (size_t)inj->n_edges, cudaMemcpyDeviceToDevice, s));
          sigmoid_kernel<<<c->sm_count * 4, 256, 0, s>>>(c->logit, c->n_edges, c->score_out); c->launches++;
          tm.end();
        } else {
          const int L = c->hp.gnn_iters;
          auto mlp = [&](int kind, int it, bool head) {
            if (kind == kEdgeNet && c->edge_tma) launch_edge_net_tma(c, it, n_hits, head, s);
            else if (kind == kEdgeEnc && c->edge_tma && c->hp.edge_enc_input == 0 && !head) launch_edge_enc_tma(c, n_hits, false, s);
            else if (kind == kEdgeEnc && c->edge_tma && c->hp.edge_enc_input == 1) launch_edge_enc_h_tma(c, n_hits, head, s);
            else if (kind == kNodeEnc && c->edge_tma) launch_edge_enc_tma(c, n_hits, true, s);
            else if (tensor_engine && c->precision == ETX_BF16 && c->engine != ETX_ENGINE_TC_SERIAL) launch_gnn_mlp_ws(c, kind, it, n_hits, head, s);
            else if (kind == kEdgeNet && c->edge_i8) launch_edge_net_i8(c, it, n_hits, head, s);
            else if (kind == kNodeNet && c->edge_i8) launch_node_net_i8(c, it, n_hits, s);
            else if (tensor_engine) launch_gnn_mlp_umma(c, kind, it, n_hits, head, s);
            else launch_gnn_mlp_simt(c, kind, it, n_hits, head, s);
          };
          tm.begin(4);
          mlp(kNodeEnc, 0, false);
          mlp(kEdgeEnc, 0, L == 0);
          tm.end();
          for (int it = 0; it < L; ++it) {
            tm.begin(5); launch_scatter(c, n_hits, s); tm.end();
            tm.begin(6); mlp(kNodeNet, it, false); tm.end();
            tm.begin(7); mlp(kEdgeNet, it, it == L - 1); tm.end();
          }
        }
      }
      if (last >= 5) {
        tm.begin(8);
        launch_components(c, c->logit, n_events, n_hits, s);
        tm.end();
      }
    }
    if (!edges_marked) {
      ETX_CUDA(cudaMemcpyAsync(c->h_n_edges_cur ? c->h_n_edges_cur : c->h_n_edges, c->n_edges, sizeof(int32_t), cudaMemcpyDeviceToHost, s));
      ETX_CUDA(cudaEventRecord(c->edges_ready_cur ? c->edges_ready_cur : c->edges_ready, s));
    }
    if (c->hp.validate_input) {     // the verdict of THIS batch: readable through etx_input_status once the stream is synchronised
      ETX_CUDA(cudaMemcpyAsync(c->h_flags_cur ? c->h_flags_cur : c->h_flags, c->flags, sizeof(int32_t), cudaMemcpyDeviceToHost, s));
      ETX_CUDA(cudaMemsetAsync(c->flags, 0, sizeof(int32_t), s));
    }
    ETX_CUDA(cudaGetLastError());
  } catch (const CudaFail& f) {
    return fail(c, ETX_ERR_CUDA, std::string(f.what) + ": " + cudaGetErrorString(f.err));
  }
  out->d_edge_src = c->src; out->d_edge_dst = c->dst; out->d_edge_score = c->score; out->d_edge_logit = c->logit;
  out->d_track_id = c->track_id; out->d_n_edges = c->n_edges; out->h_n_edges = c->h_n_edges; out->n_hits = n_hits;
  return ETX_OK;
}

}  // namespace

namespace etx {
void* etx_device_alloc(etx_ctx* c, size_t bytes) {
  void* p = nullptr;
  if (c->hp.alloc) {
    p = c->hp.alloc(bytes, c->hp.alloc_ctx);
    if (p && (reinterpret_cast<uintptr_t>(p) & 255u)) {      // contract: 256-byte alignment (TMA, 16-byte vector access)
      if (c->hp.dealloc) c->hp.dealloc(p, c->hp.alloc_ctx);
      c->error = "alloc callback returned memory that is not aligned to 256 bytes";
      return nullptr;
    }
  } else if (cudaMalloc(&p, bytes) != cudaSuccess) {
    (void)cudaGetLastError();
    p = nullptr;
  }
  if (!p) return nullptr;
  c->allocs.push_back(p);
  c->device_bytes += bytes;
  return p;
}
}  // namespace etx

extern "C" {

etx_status etx_create(const void* blob, size_t blob_bytes, const etx_hyperparams* hp, etx_handle* out) {
  if (!blob || !hp || !out) return ETX_ERR_ARG;
  if (hp->struct_size != sizeof(etx_hyperparams)) return ETX_ERR_ARG;
  etx_ctx* c = new (std::nothrow) etx_ctx();
  if (!c) return ETX_ERR_CUDA;
  c->hp = *hp;
  c->precision = hp->precision; c->engine = hp->engine;
  auto bail = [&](etx_status st) { etx_destroy(c); return st; };
  if (hp->precision < 0 || hp->precision > 2 || hp->engine < 0 || hp->engine > 2) return bail(ETX_ERR_ARG);
  if ((hp->alloc == nullptr) != (hp->dealloc == nullptr)) return bail(ETX_ERR_ARG);
  if (hp->n_planes < 1 || hp->n_planes > 1024 || hp->k < 1 || hp->window < 1 || hp->max_events < 0 || hp->max_hits < 0 ||
      hp->gnn_iters < 0 || hp->gnn_iters > 64 || hp->max_triplets < 0 || !(hp->triplet_threshold >= 0.0f && hp->triplet_threshold <= 1.0f) || hp->emb_n_hidden_layers < 1 || hp->emb_n_hidden_layers > 8 ||
      !(hp->threshold >= 0.0f && hp->threshold <= 1.0f) || isnan(hp->d2_max))
    return bail(ETX_ERR_ARG);
  for (int i = 0; i < 3; ++i)
    if (!(hp->norm_div[i] != 0.0f) || (hp->emb_input && !(hp->cyl_div[i] != 0.0f))) return bail(ETX_ERR_ARG);
  // shapes built into the kernels
  if (!(hp->emb_hidden == 64 || hp->emb_hidden == 128) || hp->emb_dim != 4 || !(hp->gnn_latent == 32 || hp->gnn_latent == 64) ||
      hp->k > 64 || (hp->edge_enc_input != 0 && hp->edge_enc_input != 1) ||
      (hp->emb_input != 0 && hp->emb_input != 1))
    return bail(ETX_ERR_UNSUPPORTED);
  if ((long long)hp->k * hp->max_hits > 0x7fffffffLL) return bail(ETX_ERR_CAPACITY);
  c->max_edges = hp->k * hp->max_hits;
  if (hp->state_dtype < 0 || hp->state_dtype > 2) return bail(ETX_ERR_ARG);
  if ((hp->precision == ETX_FP32 && hp->state_dtype == ETX_STATE_BF16) || (hp->precision == ETX_BF16 && hp->state_dtype == ETX_STATE_FP32))
    return bail(ETX_ERR_UNSUPPORTED);
  c->state_bf16 = (hp->precision == ETX_BF16) || (hp->precision == ETX_INT8 && hp->state_dtype == ETX_STATE_BF16);
  if (hp->threshold <= 0.0f) c->tau = -INFINITY;
  else if (hp->threshold >= 1.0f) c->tau = INFINITY;
  else c->tau = (float)log((double)hp->threshold / (1.0 - (double)hp->threshold));      // R17
  if (hp->triplet_threshold <= 0.0f) c->tau_t = -INFINITY;
  else if (hp->triplet_threshold >= 1.0f) c->tau_t = INFINITY;
  else c->tau_t = (float)log((double)hp->triplet_threshold / (1.0 - (double)hp->triplet_threshold));
  etx_status st = ETX_OK;
  try {
    st = parse_blob(c, static_cast<const uint8_t*>(blob), blob_bytes);
  } catch (const std::bad_alloc&) {
    c->error = "out of host memory while parsing the blob";
    return bail(ETX_ERR_BLOB);
  }
  if (st != ETX_OK) return bail(st);
  try {
    int dev = 0;
    ETX_CUDA(cudaGetDevice(&dev));
    c->device = dev;
    ETX_CUDA(cudaDeviceGetAttribute(&c->sm_count, cudaDevAttrMultiProcessorCount, dev));
    for (auto& l : c->layers) convert_layer(c, l);
    const size_t N = (size_t)hp->max_hits, E = (size_t)c->max_edges, B = (size_t)hp->max_events, d = hp->gnn_latent;
    const size_t sb = c->state_bf16 ? 2 : 4;
    c->event_off = dev_alloc<int32_t>(c, B + 1);
    c->plane_off = dev_alloc<int32_t>(c, B * (hp->n_planes + 1));
    c->knn_redo = dev_alloc<int32_t>(c, B * hp->n_planes + 1);
    c->feat = dev_alloc<float4>(c, N);
    c->feat_emb = hp->emb_input ? dev_alloc<float4>(c, N) : c->feat;
    c->emb = dev_alloc<float4>(c, N);
    c->nbr = dev_alloc<int32_t>(c, N * hp->k);
    c->deg = dev_alloc<int32_t>(c, N);
    c->row_ptr = dev_alloc<int32_t>(c, N + 1);
    c->col_ptr = dev_alloc<int32_t>(c, N + 1);
    c->cursor = dev_alloc<int32_t>(c, N + 1);
    c->src = dev_alloc<int32_t>(c, E);
    c->dst = dev_alloc<int32_t>(c, E);
    c->in_edge = dev_alloc<int32_t>(c, E);
    c->scan_tmp = dev_alloc<int32_t>(c, N / 2048 + 2);
    c->n_edges = dev_alloc<int32_t>(c, 1);
    c->flags = dev_alloc<int32_t>(c, 1);
    c->h = dev_alloc<uint8_t>(c, N * d * sb + 256);
    c->m = dev_alloc<uint8_t>(c, N * 2 * d * sb + 256);
    c->e = dev_alloc<uint8_t>(c, E * d * sb + 256);
    c->logit = dev_alloc<float>(c, E);
    c->score = dev_alloc<float>(c, E);
    c->score_out = c->score;
    c->track_id = dev_alloc<int32_t>(c, N);
    c->trk_size = dev_alloc<int32_t>(c, N); c->trk_keep = dev_alloc<int32_t>(c, N + 1);
    c->trk_number = dev_alloc<int32_t>(c, N + 1); c->trk_ksize = dev_alloc<int32_t>(c, N + 1);
    c->trk_index = dev_alloc<int32_t>(c, N); c->trk_offsets = dev_alloc<int32_t>(c, N + 1);
    c->trk_hits = dev_alloc<int32_t>(c, N); c->trk_event_off = dev_alloc<int32_t>(c, B + 1);
    c->n_tracks = dev_alloc<int32_t>(c, 1);
    if (hp->max_triplets > 0) {
      const size_t T = (size_t)hp->max_triplets;
      c->trip_cnt = dev_alloc<int32_t>(c, 3 * (N + 1)); c->trip_off = dev_alloc<int32_t>(c, 3 * (N + 1));
      c->trip_first = dev_alloc<int32_t>(c, 3 * T); c->trip_second = dev_alloc<int32_t>(c, 3 * T); c->trip_hit = dev_alloc<int32_t>(c, 3 * T);
      c->trip_logit = dev_alloc<float>(c, 3 * T); c->trip_score = dev_alloc<float>(c, 3 * T);
      c->trip_total = dev_alloc<int32_t>(c, 4);
      c->tc_par1 = dev_alloc<int32_t>(c, E); c->tc_par2 = dev_alloc<int32_t>(c, E);
      c->tc_succ = dev_alloc<int32_t>(c, E); c->tc_pred = dev_alloc<int32_t>(c, E); c->tc_comp = dev_alloc<int32_t>(c, E);
      c->tc_shared = dev_alloc<int32_t>(c, 2 * T);
      c->tc_tab_size = 1024; while (c->tc_tab_size < 2 * T) c->tc_tab_size <<= 1;
      c->tc_tab = dev_alloc<unsigned long long>(c, c->tc_tab_size);
      c->tc_n_shared = dev_alloc<int32_t>(c, 1);
      ETX_CUDA(cudaMemset(c->tc_n_shared, 0, sizeof(int32_t)));
      ETX_CUDA(cudaMallocHost(&c->h_tc_n_shared, sizeof(int32_t)));
      c->h_tc_n_shared[0] = 0;
      // etx_triplet_tracks: a hit is listed once per set it touches (at most once per kept incident edge: 2 E in all)
      c->tt_set_off = dev_alloc<int32_t>(c, E + 1);
      c->tt_set_hits = dev_alloc<int32_t>(c, 2 * E);
      c->tt_bucket_cand = dev_alloc<int32_t>(c, T + E);
      c->tt_scan_tmp = dev_alloc<int32_t>(c, (E > N ? E : N) / 2048 + 2);
      // at most one track per shared articulation plus one per set of connected edges: T + E can never overflow; the
      // listed hits have no such bound (a shared set is listed once per articulation that shares it)
      c->tt_track_cap = (int)std::min<size_t>(T + E, 0x7ffffff0);
      c->tt_hit_cap = (int)std::min<size_t>(2 * (T + E), 0x7ffffff0);
      c->tt_track_len = dev_alloc<int32_t>(c, (size_t)c->tt_track_cap + 1);
      c->tt_track_off = dev_alloc<int32_t>(c, (size_t)c->tt_track_cap + 1);
      c->tt_track_hits = dev_alloc<int32_t>(c, (size_t)c->tt_hit_cap);
      c->tt_counts = dev_alloc<int32_t>(c, 4);
      ETX_CUDA(cudaMemset(c->tt_counts, 0, 4 * sizeof(int32_t)));
      ETX_CUDA(cudaMemset(c->tt_track_off, 0, sizeof(int32_t)));
      ETX_CUDA(cudaMallocHost(&c->h_tt_counts, 4 * sizeof(int32_t)));
      for (int i = 0; i < 4; ++i) c->h_tt_counts[i] = 0;
      ETX_CUDA(cudaMemset(c->trip_total, 0, 4 * sizeof(int32_t)));
      ETX_CUDA(cudaMallocHost(&c->h_trip_total, 4 * sizeof(int32_t)));
      for (int i = 0; i < 4; ++i) c->h_trip_total[i] = 0;
    }
    c->d_xyz_in = dev_alloc<float>(c, N * 3);
    c->d_plane_in = dev_alloc<int32_t>(c, N);
    ETX_CUDA(cudaMemset(c->n_edges, 0, sizeof(int32_t)));
    ETX_CUDA(cudaMemset(c->flags, 0, sizeof(int32_t)));
    ETX_CUDA(cudaMallocHost(&c->h_event_off, sizeof(int32_t) * (B + 1)));
    ETX_CUDA(cudaMallocHost(&c->h_n_edges, sizeof(int32_t)));
    ETX_CUDA(cudaMallocHost(&c->h_n_tracks, sizeof(int32_t)));
    c->h_n_tracks[0] = 0;
    ETX_CUDA(cudaMallocHost(&c->h_flags, sizeof(int32_t)));
    c->h_n_edges[0] = 0; c->h_flags[0] = 0;
    ETX_CUDA(cudaEventCreateWithFlags(&c->staging_free, cudaEventDisableTiming));
    ETX_CUDA(cudaEventCreateWithFlags(&c->edges_ready, cudaEventDisableTiming));
    ETX_CUDA(cudaEventCreateWithFlags(&c->copies_done, cudaEventDisableTiming));
    ETX_CUDA(cudaStreamCreateWithFlags(&c->copy_stream, cudaStreamNonBlocking));
    for (int i = 0; i < 256; ++i) ETX_CUDA(cudaEventCreate(&c->ev[i]));
    simt_configure(c);
    if (c->precision != ETX_FP32 && c->engine != ETX_ENGINE_SIMT) {
      if (!umma_supported(c)) { c->error = "tensor-core engine not available for these shapes"; return bail(ETX_ERR_UNSUPPORTED); }
      umma_configure(c);
      if (c->precision == ETX_INT8 && c->engine == ETX_ENGINE_AUTO) {
        if (!edge_i8_configure(c)) { c->error = "INT8 edge-network TMA setup failed"; return bail(ETX_ERR_CUDA); }
        c->edge_i8 = true;
      }
      if (c->precision == ETX_BF16 && c->engine == ETX_ENGINE_AUTO) {
        if (!edge_tma_configure(c)) { c->error = "edge-network TMA setup failed"; return bail(ETX_ERR_CUDA); }
        c->edge_tma = true;
      }
    }
    ETX_CUDA(cudaDeviceSynchronize());
  } catch (const CudaFail& f) {
    (void)f;
    return bail(ETX_ERR_CUDA);
  } catch (const std::bad_alloc&) {
    return bail(ETX_ERR_CUDA);
  }
  *out = c;
  return ETX_OK;
}

etx_status etx_destroy(etx_handle c) {
  if (!c) return ETX_OK;
  cudaDeviceSynchronize();
  for (void* p : c->allocs) { if (c->hp.alloc) { if (c->hp.dealloc) c->hp.dealloc(p, c->hp.alloc_ctx); } else cudaFree(p); }
  if (c->h_event_off) cudaFreeHost(c->h_event_off);
  if (c->h_n_edges) cudaFreeHost(c->h_n_edges);
  if (c->h_n_tracks) cudaFreeHost(c->h_n_tracks);
  if (c->h_flags) cudaFreeHost(c->h_flags);
  if (c->h_trip_total) cudaFreeHost(c->h_trip_total);
  if (c->h_tc_n_shared) cudaFreeHost(c->h_tc_n_shared);
  if (c->h_tt_counts) cudaFreeHost(c->h_tt_counts);
  if (c->h_slot_flags) cudaFreeHost(c->h_slot_flags);
  if (c->h_slot_n_edges) cudaFreeHost(c->h_slot_n_edges);
  for (int i = 0; i < 2; ++i) {
    if (c->slot_edges_ready[i]) cudaEventDestroy(c->slot_edges_ready[i]);
    if (c->slot_edges_copied[i]) cudaEventDestroy(c->slot_edges_copied[i]);
    if (c->slot_copies_done[i]) cudaEventDestroy(c->slot_copies_done[i]);
    if (c->slot_done[i]) cudaEventDestroy(c->slot_done[i]);
    if (c->slot_inputs_read[i]) cudaEventDestroy(c->slot_inputs_read[i]);
    if (c->slot_h2d[i]) cudaEventDestroy(c->slot_h2d[i]);
  }
  if (c->staging_free) cudaEventDestroy(c->staging_free);
  if (c->edges_ready) cudaEventDestroy(c->edges_ready);
  if (c->copies_done) cudaEventDestroy(c->copies_done);
  if (c->copy_stream) cudaStreamDestroy(c->copy_stream);
  if (c->h2d_stream) cudaStreamDestroy(c->h2d_stream);
  for (int i = 0; i < 256; ++i) if (c->ev[i]) cudaEventDestroy(c->ev[i]);
  delete c;
  return ETX_OK;
}

etx_status etx_run(etx_handle c, const float* d_xyz, const int32_t* d_plane, const int32_t* h_event_offsets,
                   int32_t n_events, etx_stream stream, etx_output* out) {
  if (c && (c->slot_unwaited[0] || c->slot_unwaited[1]))
    return fail(c, ETX_ERR_ARG, "a submission of etx_submit_host has not been waited for yet (etx_wait_host)");
  return run_impl(c, d_xyz, d_plane, h_event_offsets, n_events, static_cast<cudaStream_t>(stream), nullptr, out);
}

etx_status etx_tracks(etx_handle c, int32_t min_hits, etx_stream stream, etx_tracks_output* out) {
  if (!c) return ETX_ERR_ARG;
  if (!out || min_hits < 1) return fail(c, ETX_ERR_ARG, "etx_tracks: null output or min_hits < 1");
  cudaStream_t s = static_cast<cudaStream_t>(stream);
  launch_tracks(c, c->last_n_events, c->last_n_hits, min_hits, s);
  if (cudaMemcpyAsync(c->h_n_tracks, c->n_tracks, sizeof(int32_t), cudaMemcpyDeviceToHost, s) != cudaSuccess ||
      cudaGetLastError() != cudaSuccess)
    return fail(c, ETX_ERR_CUDA, "etx_tracks: launch failed");
  out->d_track_index = c->trk_index; out->d_track_offsets = c->trk_offsets; out->d_track_hits = c->trk_hits;
  out->d_event_track_offsets = c->trk_event_off; out->d_n_tracks = c->n_tracks; out->h_n_tracks = c->h_n_tracks;
  return ETX_OK;
}

etx_status etx_triplets(etx_handle c, etx_stream stream, etx_triplets_output* out) {
  if (!c) return ETX_ERR_ARG;
  if (!out) return fail(c, ETX_ERR_ARG, "etx_triplets: null output");
  if (c->i_trip < 0) return fail(c, ETX_ERR_BLOB, "etx_triplets: the blob carries no triplet classifiers (header word 11)");
  if (c->hp.max_triplets <= 0) return fail(c, ETX_ERR_CAPACITY, "etx_triplets: max_triplets is 0");
  cudaStream_t s = static_cast<cudaStream_t>(stream);
  launch_triplet_build(c, c->last_n_hits, s);
  for (int k = 0; k < 3; ++k) launch_triplet_classifier(c, k, s);
  if (cudaMemcpyAsync(c->h_trip_total, c->trip_total, 3 * sizeof(int32_t), cudaMemcpyDeviceToHost, s) != cudaSuccess ||
      cudaGetLastError() != cudaSuccess)
    return fail(c, ETX_ERR_CUDA, "etx_triplets: launch failed");
  const size_t T = (size_t)c->hp.max_triplets;
  for (int k = 0; k < 3; ++k) {
    out->d_first[k] = c->trip_first + k * T; out->d_second[k] = c->trip_second + k * T; out->d_hit[k] = c->trip_hit + k * T;
    out->d_logit[k] = c->trip_logit + k * T; out->d_score[k] = c->trip_score + k * T;
  }
  out->d_count = c->trip_total; out->h_count = c->h_trip_total; out->capacity = c->hp.max_triplets;
  return ETX_OK;
}

etx_status etx_triplet_components(etx_handle c, etx_stream stream, etx_triplet_components_output* out) {
  if (!c) return ETX_ERR_ARG;
  if (!out) return fail(c, ETX_ERR_ARG, "etx_triplet_components: null output");
  if (c->i_trip < 0 || c->hp.max_triplets <= 0) return fail(c, ETX_ERR_CAPACITY, "etx_triplet_components: the triplet stage is not configured");
  cudaStream_t s = static_cast<cudaStream_t>(stream);
  launch_triplet_components(c, s);
  if (cudaMemcpyAsync(c->h_tc_n_shared, c->tc_n_shared, sizeof(int32_t), cudaMemcpyDeviceToHost, s) != cudaSuccess ||
      cudaGetLastError() != cudaSuccess)
    return fail(c, ETX_ERR_CUDA, "etx_triplet_components: launch failed");
  out->d_edge_component = c->tc_comp; out->d_shared = c->tc_shared; out->d_n_shared = c->tc_n_shared;
  out->h_n_shared = c->h_tc_n_shared; out->capacity = c->hp.max_triplets;
  return ETX_OK;
}

etx_status etx_calibrate(etx_handle c, const float* d_xyz, const int32_t* d_plane, const int32_t* h_event_offsets, int32_t n_events,
                         etx_stream stream, float* h_scales, int32_t capacity, int32_t* n_scales) {
  if (!c) return ETX_ERR_ARG;
  if (!n_scales) return fail(c, ETX_ERR_ARG, "etx_calibrate: null n_scales");
  int nq = 0;
  for (auto& l : c->layers) nq += l.tensor;
  *n_scales = nq;
  if (!h_scales) return ETX_OK;                              // query: how many scales the model needs
  if (capacity < nq) return fail(c, ETX_ERR_CAPACITY, "etx_calibrate: h_scales is too small (see *n_scales)");
  if (c->precision != ETX_FP32)
    return fail(c, ETX_ERR_UNSUPPORTED, "etx_calibrate records the fp32 forward: create the handle with precision ETX_FP32");
  if (c->slot_unwaited[0] || c->slot_unwaited[1])
    return fail(c, ETX_ERR_ARG, "a submission of etx_submit_host has not been waited for yet (etx_wait_host)");
  if (c->i_trip >= 0 && c->hp.max_triplets <= 0)
    return fail(c, ETX_ERR_CAPACITY, "etx_calibrate: the blob carries triplet classifiers; set max_triplets so that their inputs can be recorded");
  cudaStream_t s = static_cast<cudaStream_t>(stream);
  const size_t nl = c->layers.size();
  std::vector<float> amax(nl, 0.0f);
  try {
    if (!c->absmax) c->absmax = dev_alloc<float>(c, nl);      // through the handle's allocator; adds to etx_workspace_bytes
    ETX_CUDA(cudaMemsetAsync(c->absmax, 0, nl * sizeof(float), s));
    c->calibrating = true;
    etx_output o;
    etx_status st = run_impl(c, d_xyz, d_plane, h_event_offsets, n_events, s, nullptr, &o);
    if (st == ETX_OK && c->i_trip >= 0) {
      launch_triplet_build(c, c->last_n_hits, s);
      for (int k = 0; k < 3; ++k) launch_triplet_classifier(c, k, s);
      ETX_CUDA(cudaMemcpyAsync(c->h_trip_total, c->trip_total, 3 * sizeof(int32_t), cudaMemcpyDeviceToHost, s));
    }
    c->calibrating = false;
    if (st != ETX_OK) return st;
    ETX_CUDA(cudaMemcpyAsync(amax.data(), c->absmax, nl * sizeof(float), cudaMemcpyDeviceToHost, s));
    ETX_CUDA(cudaStreamSynchronize(s));
    ETX_CUDA(cudaGetLastError());
  } catch (const CudaFail& f) {
    c->calibrating = false;
    return fail(c, ETX_ERR_CUDA, std::string(f.what) + ": " + cudaGetErrorString(f.err));
  }
  if (etx_input_status(c) != ETX_OK) return ETX_ERR_INPUT_ORDER;
  if (c->i_trip >= 0)
    for (int k = 0; k < 3; ++k)
      if (c->h_trip_total[k] > c->hp.max_triplets)
        return fail(c, ETX_ERR_CAPACITY, "etx_calibrate: more triplets than max_triplets; the triplet classifiers saw only a part of their inputs");
  int q = 0;
  for (auto& l : c->layers)
    if (l.tensor) { const float a = amax[l.index]; h_scales[q++] = a > 0.0f ? a / 127.0f : 1.0f; }
  return ETX_OK;
}

etx_status etx_triplet_tracks(etx_handle c, int32_t min_hits, etx_stream stream, etx_triplet_tracks_output* out) {
  if (!c) return ETX_ERR_ARG;
  if (!out || min_hits < 1) return fail(c, ETX_ERR_ARG, "etx_triplet_tracks: null output or min_hits < 1");
  if (c->i_trip < 0 || c->hp.max_triplets <= 0) return fail(c, ETX_ERR_CAPACITY, "etx_triplet_tracks: the triplet stage is not configured");
  if ((long long)c->hp.max_triplets + c->max_edges > 0x7fffffffLL)
    return fail(c, ETX_ERR_UNSUPPORTED, "etx_triplet_tracks: max_triplets + k * max_hits must stay below 2^31");
  cudaStream_t s = static_cast<cudaStream_t>(stream);
  launch_triplet_tracks(c, c->last_n_events, c->last_n_hits, min_hits, s);
  if (cudaMemcpyAsync(c->h_tt_counts, c->tt_counts, 4 * sizeof(int32_t), cudaMemcpyDeviceToHost, s) != cudaSuccess ||
      cudaGetLastError() != cudaSuccess)
    return fail(c, ETX_ERR_CUDA, "etx_triplet_tracks: launch failed");
  out->d_track_offsets = c->tt_track_off; out->d_track_hits = c->tt_track_hits; out->d_counts = c->tt_counts;
  out->h_counts = c->h_tt_counts; out->track_capacity = c->tt_track_cap; out->hit_capacity = c->tt_hit_cap;
  return ETX_OK;
}

etx_status etx_dbg_run(etx_handle c, const float* d_xyz, const int32_t* d_plane, const int32_t* h_event_offsets,
                       int32_t n_events, etx_stream stream, const etx_inject* inj, etx_output* out) {
  if (c && (c->slot_unwaited[0] || c->slot_unwaited[1]))
    return fail(c, ETX_ERR_ARG, "a submission of etx_submit_host has not been waited for yet (etx_wait_host)");
  return run_impl(c, d_xyz, d_plane, h_event_offsets, n_events, static_cast<cudaStream_t>(stream), inj, out);
}

etx_status etx_run_host(etx_handle c, const float* h_xyz, const int32_t* h_plane, const int32_t* h_event_offsets,
                        int32_t n_events, etx_stream stream, float* h_edge_score, int32_t* h_edge_src,
                        int32_t* h_edge_dst, int32_t* h_track_id, int32_t* n_edges_out) {
  if (!c) return ETX_ERR_ARG;
  if (c && (c->slot_unwaited[0] || c->slot_unwaited[1]))
    return fail(c, ETX_ERR_ARG, "a submission of etx_submit_host has not been waited for yet (etx_wait_host)");
  if (!h_event_offsets || n_events < 0 || !n_edges_out) return fail(c, ETX_ERR_ARG, "null argument");
  if (n_events > c->hp.max_events) return fail(c, ETX_ERR_CAPACITY, "n_events exceeds max_events");
  const int n_hits = h_event_offsets[n_events];
  if (n_hits < 0 || n_hits > c->hp.max_hits) return fail(c, ETX_ERR_CAPACITY, "n_hits exceeds max_hits");
  if (n_hits > 0 && (!h_xyz || !h_plane)) return fail(c, ETX_ERR_ARG, "null hit arrays");
  cudaStream_t s = static_cast<cudaStream_t>(stream);
  try {
    if (n_hits > 0) {
      ETX_CUDA(cudaMemcpyAsync(c->d_xyz_in, h_xyz, sizeof(float) * 3 * (size_t)n_hits, cudaMemcpyHostToDevice, s));
      ETX_CUDA(cudaMemcpyAsync(c->d_plane_in, h_plane, sizeof(int32_t) * (size_t)n_hits, cudaMemcpyHostToDevice, s));
    }
    // Pinned (page-locked) host memory is addressable from the device: the classifier then writes the scores
    // straight into the caller's buffer while it computes, and the 4 E byte copy after the run disappears.
    bool score_direct = false;
    if (h_edge_score) {
      cudaPointerAttributes attr;
      if (cudaPointerGetAttributes(&attr, h_edge_score) == cudaSuccess && attr.type == cudaMemoryTypeHost && attr.devicePointer) {
        c->score_out = static_cast<float*>(attr.devicePointer);
        score_direct = true;
      } else {
        (void)cudaGetLastError();                              // pageable memory: not an error, take the copy path
      }
    }
    etx_output o;
    etx_status st = run_impl(c, c->d_xyz_in, c->d_plane_in, h_event_offsets, n_events, s, nullptr, &o);
    c->score_out = c->score;
    if (st != ETX_OK) return st;
    // src / dst are final after S3: their D2H copy runs on the copy stream while the GNN is still computing
    ETX_CUDA(cudaEventSynchronize(c->edges_ready));
    const int E = c->h_n_edges[0];
    *n_edges_out = E;
    if (E > 0 && (h_edge_src || h_edge_dst)) {
      ETX_CUDA(cudaStreamWaitEvent(c->copy_stream, c->edges_ready, 0));
      if (h_edge_src) ETX_CUDA(cudaMemcpyAsync(h_edge_src, c->src, sizeof(int32_t) * (size_t)E, cudaMemcpyDeviceToHost, c->copy_stream));
      if (h_edge_dst) ETX_CUDA(cudaMemcpyAsync(h_edge_dst, c->dst, sizeof(int32_t) * (size_t)E, cudaMemcpyDeviceToHost, c->copy_stream));
      ETX_CUDA(cudaEventRecord(c->copies_done, c->copy_stream));
      ETX_CUDA(cudaStreamWaitEvent(s, c->copies_done, 0));      // the caller's stream stays the single point to wait on
    }
    if (h_track_id && n_hits > 0)
      ETX_CUDA(cudaMemcpyAsync(h_track_id, c->track_id, sizeof(int32_t) * (size_t)n_hits, cudaMemcpyDeviceToHost, s));
    if (E > 0 && h_edge_score && !score_direct) ETX_CUDA(cudaMemcpyAsync(h_edge_score, c->score, sizeof(float) * (size_t)E, cudaMemcpyDeviceToHost, s));
    ETX_CUDA(cudaStreamSynchronize(s));
  } catch (const CudaFail& f) {
    return fail(c, ETX_ERR_CUDA, std::string(f.what) + ": " + cudaGetErrorString(f.err));
  }
  return etx_input_status(c);          // the stream is synchronised: the verdict of this very batch
}

etx_status etx_input_status(etx_handle c) {
  if (!c) return ETX_ERR_ARG;
  if (c->hp.validate_input && (c->h_flags[0] & 1))
    return fail(c, ETX_ERR_INPUT_ORDER, "hits not sorted by (event, plane), or a plane index out of range: the batch was rejected (0 edges)");
  return ETX_OK;
}

static void* mapped_ptr(void* host) {
  if (!host) return nullptr;
  cudaPointerAttributes attr;
  if (cudaPointerGetAttributes(&attr, host) == cudaSuccess && attr.type == cudaMemoryTypeHost && attr.devicePointer) return attr.devicePointer;
  (void)cudaGetLastError();
  return nullptr;
}

// The edge list of a submission can only be copied out once the host knows E.  That is learnt without stalling the
// pipeline: the copy of submission i is issued by the NEXT call on the handle (etx_submit_host of i + 1, or
// etx_wait_host of i), by which time S3 of batch i -- an early stage -- has long passed while its GNN still runs.
static void flush_edge_copy(etx_ctx* c, int slot) {
  etx_ctx::PendingCopy& pc = c->slot_copy[slot];
  if (!pc.pending) return;
  pc.pending = false;
  ETX_CUDA(cudaEventSynchronize(c->slot_edges_ready[slot]));
  const int E = c->h_slot_n_edges[slot];
  *pc.h_n = E;
  ETX_CUDA(cudaStreamWaitEvent(c->copy_stream, c->slot_edges_ready[slot], 0));
  if (E > 0 && pc.h_src) ETX_CUDA(cudaMemcpyAsync(pc.h_src, c->src, sizeof(int32_t) * (size_t)E, cudaMemcpyDeviceToHost, c->copy_stream));
  if (E > 0 && pc.h_dst) ETX_CUDA(cudaMemcpyAsync(pc.h_dst, c->dst, sizeof(int32_t) * (size_t)E, cudaMemcpyDeviceToHost, c->copy_stream));
  ETX_CUDA(cudaEventRecord(c->slot_edges_copied[slot], c->copy_stream));
  // the scores leave once the batch's last kernel has written them -- under the next batch's compute, from this slot's
  // own score buffer
  ETX_CUDA(cudaStreamWaitEvent(c->copy_stream, c->slot_done[slot], 0));
  if (E > 0 && pc.h_score) ETX_CUDA(cudaMemcpyAsync(pc.h_score, pc.d_score, sizeof(float) * (size_t)E, cudaMemcpyDeviceToHost, c->copy_stream));
  ETX_CUDA(cudaEventRecord(c->slot_copies_done[slot], c->copy_stream));
}

etx_status etx_submit_host(etx_handle c, const float* h_xyz, const int32_t* h_plane, const int32_t* h_event_offsets,
                           int32_t n_events, etx_stream stream, float* h_edge_score, int32_t* h_edge_src,
                           int32_t* h_edge_dst, int32_t* h_track_id, int32_t* h_n_edges, int32_t* ticket) {
  if (!c) return ETX_ERR_ARG;
  if (!h_event_offsets || n_events < 0 || !h_n_edges || !ticket) return fail(c, ETX_ERR_ARG, "null argument");
  if (n_events > c->hp.max_events) return fail(c, ETX_ERR_CAPACITY, "n_events exceeds max_events");
  const int n_hits = h_event_offsets[n_events];
  if (n_hits < 0 || n_hits > c->hp.max_hits) return fail(c, ETX_ERR_CAPACITY, "n_hits exceeds max_hits");
  if (n_hits > 0 && (!h_xyz || !h_plane)) return fail(c, ETX_ERR_ARG, "null hit arrays");
  // pinned output buffers: the copies must be truly asynchronous
  if ((h_edge_score && !mapped_ptr(h_edge_score)) || (h_edge_src && !mapped_ptr(h_edge_src)) || (h_edge_dst && !mapped_ptr(h_edge_dst)) ||
      (h_track_id && !mapped_ptr(h_track_id)))
    return fail(c, ETX_ERR_ARG, "etx_submit_host needs pinned (page-locked) output buffers");
  cudaStream_t s = static_cast<cudaStream_t>(stream);
  const int slot = (int)(c->n_submitted & 1), prev = slot ^ 1;
  try {
    if (!c->submit_ready) {
      // first use: the second staging set, the second score buffer and the per-slot events.  Every resource is created
      // only if it does not exist yet and the flag is set last, so a call that failed half-way is completed by the next
      // one instead of leaving null events behind.  (These blocks add to etx_workspace_bytes.)
      if (!c->d_xyz_in2) c->d_xyz_in2 = dev_alloc<float>(c, (size_t)c->hp.max_hits * 3);
      if (!c->d_plane_in2) c->d_plane_in2 = dev_alloc<int32_t>(c, (size_t)c->hp.max_hits);
      if (!c->score2) c->score2 = dev_alloc<float>(c, (size_t)c->max_edges);
      if (!c->h2d_stream) ETX_CUDA(cudaStreamCreateWithFlags(&c->h2d_stream, cudaStreamNonBlocking));
      if (!c->h_slot_flags) { ETX_CUDA(cudaMallocHost(&c->h_slot_flags, 2 * sizeof(int32_t))); c->h_slot_flags[0] = c->h_slot_flags[1] = 0; }
      if (!c->h_slot_n_edges) { ETX_CUDA(cudaMallocHost(&c->h_slot_n_edges, 2 * sizeof(int32_t))); c->h_slot_n_edges[0] = c->h_slot_n_edges[1] = 0; }
      for (int i = 0; i < 2; ++i)
        for (cudaEvent_t* ev : {&c->slot_done[i], &c->slot_inputs_read[i], &c->slot_h2d[i], &c->slot_edges_ready[i],
                                &c->slot_copies_done[i], &c->slot_edges_copied[i]})
          if (!*ev) ETX_CUDA(cudaEventCreateWithFlags(ev, cudaEventDisableTiming));
      c->submit_ready = true;
    }
    // Submission i - 2 used this slot: its results (validation verdict, E, device score buffer, the caller's output
    // buffers) are released by etx_wait_host and by nothing else -- the edge-list copy that submission i - 1 issued on
    // its behalf does not count.
    if (c->slot_unwaited[slot]) return fail(c, ETX_ERR_ARG, "etx_submit_host: wait for submission i before submitting i + 2");
    // belt and braces for the slot's score buffer: this batch's classifier must not write it before the D2H of the
    // scores of submission i - 2 has finished (etx_wait_host has synchronised on that event already)
    if (c->n_submitted >= 2) ETX_CUDA(cudaStreamWaitEvent(s, c->slot_copies_done[slot], 0));
    // the previous submission's edge list: issue its copy now, and keep this batch's S3 from overwriting src / dst early
    if (c->n_submitted >= 1) {
      flush_edge_copy(c, prev);
      ETX_CUDA(cudaStreamWaitEvent(s, c->slot_edges_copied[prev], 0));
    }
    float* dx = slot ? c->d_xyz_in2 : c->d_xyz_in;
    int32_t* dp = slot ? c->d_plane_in2 : c->d_plane_in;
    // H2D on its own stream, under the previous batch's compute; the staging set was last read by S0 two submissions ago
    if (c->n_submitted >= 2) ETX_CUDA(cudaStreamWaitEvent(c->h2d_stream, c->slot_inputs_read[slot], 0));
    if (n_hits > 0) {
      ETX_CUDA(cudaMemcpyAsync(dx, h_xyz, sizeof(float) * 3 * (size_t)n_hits, cudaMemcpyHostToDevice, c->h2d_stream));
      ETX_CUDA(cudaMemcpyAsync(dp, h_plane, sizeof(int32_t) * (size_t)n_hits, cudaMemcpyHostToDevice, c->h2d_stream));
    }
    ETX_CUDA(cudaEventRecord(c->slot_h2d[slot], c->h2d_stream));
    ETX_CUDA(cudaStreamWaitEvent(s, c->slot_h2d[slot], 0));
    c->score_out = slot ? c->score2 : c->score;
    c->h_flags_cur = &c->h_slot_flags[slot];
    c->inputs_read_cur = c->slot_inputs_read[slot];
    c->edges_ready_cur = c->slot_edges_ready[slot];
    c->h_n_edges_cur = &c->h_slot_n_edges[slot];
    etx_output o;
    const etx_status st = run_impl(c, dx, dp, h_event_offsets, n_events, s, nullptr, &o);
    c->score_out = c->score; c->h_flags_cur = nullptr; c->inputs_read_cur = nullptr; c->edges_ready_cur = nullptr; c->h_n_edges_cur = nullptr;
    if (st != ETX_OK) return st;
    if (h_track_id && n_hits > 0)
      ETX_CUDA(cudaMemcpyAsync(h_track_id, c->track_id, sizeof(int32_t) * (size_t)n_hits, cudaMemcpyDeviceToHost, s));
    ETX_CUDA(cudaEventRecord(c->slot_done[slot], s));
    c->slot_copy[slot].h_src = h_edge_src; c->slot_copy[slot].h_dst = h_edge_dst; c->slot_copy[slot].h_n = h_n_edges;
    c->slot_copy[slot].h_score = h_edge_score; c->slot_copy[slot].d_score = slot ? c->score2 : c->score;
    c->slot_copy[slot].pending = true;
    c->slot_unwaited[slot] = true;
    ETX_CUDA(cudaGetLastError());
  } catch (const CudaFail& f) {
    return fail(c, ETX_ERR_CUDA, std::string(f.what) + ": " + cudaGetErrorString(f.err));
  }
  *ticket = (int32_t)(c->n_submitted & 0x7fffffff);
  c->n_submitted++;
  return ETX_OK;
}

etx_status etx_wait_host(etx_handle c, int32_t ticket) {
  if (!c) return ETX_ERR_ARG;
  const long long newest = (c->n_submitted - 1) & 0x7fffffff;
  const long long t = (long long)ticket;
  if (c->n_submitted == 0 || t > newest || newest - t > 1)
    return fail(c, ETX_ERR_ARG, "etx_wait_host: unknown ticket (only the last two submissions can be waited for)");
  const int slot = (int)(t & 1);
  try {
    flush_edge_copy(c, slot);
    ETX_CUDA(cudaEventSynchronize(c->slot_copies_done[slot]));
    ETX_CUDA(cudaEventSynchronize(c->slot_done[slot]));
  } catch (const CudaFail& f) {
    return fail(c, ETX_ERR_CUDA, std::string(f.what) + ": " + cudaGetErrorString(f.err));
  }
  c->slot_unwaited[slot] = false;
  if (c->hp.validate_input && (c->h_slot_flags[slot] & 1))
    return fail(c, ETX_ERR_INPUT_ORDER, "hits not sorted by (event, plane), or a plane index out of range: the batch was rejected (0 edges)");
  return ETX_OK;
}

const char* etx_status_string(etx_status s) {
  switch (s) {
    case ETX_OK: return "ETX_OK";
    case ETX_ERR_ARG: return "ETX_ERR_ARG";
    case ETX_ERR_BLOB: return "ETX_ERR_BLOB";
    case ETX_ERR_CAPACITY: return "ETX_ERR_CAPACITY";
    case ETX_ERR_INPUT_ORDER: return "ETX_ERR_INPUT_ORDER";
    case ETX_ERR_CUDA: return "ETX_ERR_CUDA";
    case ETX_ERR_UNSUPPORTED: return "ETX_ERR_UNSUPPORTED";
  }
  return "ETX_ERR_UNKNOWN";
}

const char* etx_last_error(etx_handle c) { return c ? c->error.c_str() : "null handle"; }

size_t etx_workspace_bytes(etx_handle c) { return c ? c->device_bytes : 0; }

etx_status etx_dbg_buffer(etx_handle c, const char* name, const void** d_ptr, size_t* bytes) {
  if (!c || !name || !d_ptr || !bytes) return ETX_ERR_ARG;
  const size_t N = (size_t)c->last_n_hits, E = (size_t)c->h_n_edges[0], d = c->hp.gnn_latent, sb = c->state_bf16 ? 2 : 4;
  const std::string n(name);
  if (n == "plane_off") { *d_ptr = c->plane_off; *bytes = (size_t)c->last_n_events * (c->hp.n_planes + 1) * 4; return ETX_OK; }
  if (n == "emb") { *d_ptr = c->emb; *bytes = N * 16; return ETX_OK; }
  if (n == "feat") { *d_ptr = c->feat; *bytes = N * 16; return ETX_OK; }
  if (n == "feat_emb") { *d_ptr = c->feat_emb; *bytes = N * 16; return ETX_OK; }
  if (n == "nbr") { *d_ptr = c->nbr; *bytes = N * c->hp.k * 4; return ETX_OK; }
  if (n == "deg") { *d_ptr = c->deg; *bytes = N * 4; return ETX_OK; }
  if (n == "row_ptr") { *d_ptr = c->row_ptr; *bytes = (N + 1) * 4; return ETX_OK; }
  if (n == "col_ptr") { *d_ptr = c->col_ptr; *bytes = (N + 1) * 4; return ETX_OK; }
  if (n == "in_edge") { *d_ptr = c->in_edge; *bytes = E * 4; return ETX_OK; }
  if (n == "h") { *d_ptr = c->h; *bytes = N * d * sb; return ETX_OK; }
  if (n == "m") { *d_ptr = c->m; *bytes = N * 2 * d * sb; return ETX_OK; }
  if (n == "e") { *d_ptr = c->e; *bytes = E * d * sb; return ETX_OK; }
  if (n == "logit") { *d_ptr = c->logit; *bytes = E * 4; return ETX_OK; }
  if (n == "tap") { *d_ptr = c->tap; *bytes = c->tap_bytes; return ETX_OK; }
  if (n == "trip_logit") { *d_ptr = c->trip_logit; *bytes = c->trip_logit ? 3 * (size_t)c->hp.max_triplets * 4 : 0; return ETX_OK; }
  return fail(c, ETX_ERR_ARG, "unknown buffer name");
}

etx_status etx_dbg_tap_layer(etx_handle c, int32_t layer_index) {
  if (!c) return ETX_ERR_ARG;
  if (layer_index < 0) { c->tap_layer = -1; return ETX_OK; }
  if (c->precision != ETX_INT8 || layer_index >= (int)c->layers.size() || !c->layers[layer_index].tensor)
    return fail(c, ETX_ERR_ARG, "tap: INT8 mode and a quantised layer index are required");
  if (!c->tap) {
    const size_t rows = (size_t)(c->max_edges > c->hp.max_hits ? c->max_edges : c->hp.max_hits);
    const size_t width = (size_t)(c->hp.emb_hidden > c->hp.gnn_latent ? c->hp.emb_hidden : c->hp.gnn_latent);
    const size_t bytes = rows * width * 4;
    if (bytes > (size_t)4 << 30) return fail(c, ETX_ERR_CAPACITY, "tap buffer would exceed 4 GiB; use a smaller max_hits");
    c->tap = static_cast<int32_t*>(etx::etx_device_alloc(c, bytes ? bytes : 4));   // through the handle's allocator, freed by etx_destroy
    if (!c->tap) return fail(c, ETX_ERR_CUDA, "tap buffer allocation failed");
    c->tap_bytes = bytes;
  }
  c->tap_layer = layer_index;
  return ETX_OK;
}

etx_status etx_dbg_enable_timing(etx_handle c, int32_t on) {
  if (!c) return ETX_ERR_ARG;
  c->timing = on != 0;
  return ETX_OK;
}

etx_status etx_dbg_stage_times(etx_handle c, float* ms_out) {
  if (!c || !ms_out) return ETX_ERR_ARG;
  for (int i = 0; i < ETX_N_STAGE_TIMES; ++i) ms_out[i] = 0.0f;
  for (auto& sp : c->spans) {
    if (sp.b < 0) continue;
    float ms = 0.0f;
    if (cudaEventElapsedTime(&ms, c->ev[sp.a], c->ev[sp.b]) != cudaSuccess) return fail(c, ETX_ERR_CUDA, "cudaEventElapsedTime");
    ms_out[sp.stage] += ms;
  }
  return ETX_OK;
}

int64_t etx_dbg_launch_count(etx_handle c) { return c ? c->launches : 0; }

}  // extern "C"
