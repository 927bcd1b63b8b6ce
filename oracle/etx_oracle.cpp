// ============================================================================
// ETX4VELO hot-path ORACLE  --  TEST INFRASTRUCTURE ONLY.
//
// A plain, slow, obviously-correct CPU implementation of the five stages of
// the ETX4VELO pipeline as implemented in C++/CUDA by the paper (PAPER.md L238
// section 7: embedding inference, k-NN, GNN up to the edge classifier, WCC).  Only
// tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl
// reference legs may build, load or call this file.  It shares no code,
// header, table or helper with the CUDA path (paper_2407_12119_b200/csrc) and
// is never a fallback for it.
//
// Every function cites the passage it follows.  Where the paper is silent the
// reading is the one listed in DESIGN.md section 4 ("Readings"), numbered R1..R31.
//
// Pins (tests/test_oracle_pins.py, run with -m "not gpu"):
//   features/MLP : closed forms on hand-made weights, float64 matmul bound; cylindrical input (R27): float64
//                  hypot / atan2 within 5e-7, quadrants, axes, signed zeros
//   bf16 rounding: torch's CPU bfloat16 conversion on edge cases + random
//   int8         : numpy int64 integer matmul, hand quantiser values
//   distance     : Eq.(1) on integer embeddings
//   k-NN         : numpy brute force over all pairs, paper's replace-the-max scan
//   edges / CSC  : permutation + ordering invariants
//   scatter-sum  : dense 0/1 incidence-matrix product (Eq.(4))
//   head         : sigmoid closed forms, threshold boundary (L80)
//   components   : scipy.sparse.csgraph + BFS + the paper's plane sweeps iterated
//   tracks       : dictionary-based regrouping in Python, partition / ordering invariants, truth particles
//   bf16 GNN     : a numpy restatement with torch.bfloat16 round trips at every R20 rounding point, bit for bit,
//                  and shown to differ when any one point is dropped
//   int8 scales  : every activation scale recomputed by an independent numpy forward, bit for bit
//   triplets     : (tests/test_oracle_triplets.py) brute force over all pairs of edges, closed-form counts; the
//                  classifier against float64 / pinned-fp32 / torch-bfloat16 restatements; track building against
//                  a set + BFS formulation of the four phases, scipy components, hand-built e+e- and skipped-plane
//                  fixtures, truth particles of a noise-free event
//   The paper prints no worked numerical example, so no value
//   here is pinned to a number printed by the paper.
//
// Arithmetic hygiene (R4): every fp32 operation is one correctly rounded IEEE
// operation in the stated order: compile with -ffp-contract=off, no
// -ffast-math; fused multiply-adds are explicit std::fmaf.
// Loops over independent rows / queries are OpenMP-parallel; that changes no
// arithmetic order (each output is still produced by one sequential chain).
// ============================================================================
#include <algorithm>
#include <cmath>
#include <cstdint>
#include <cstring>
#include <limits>
#include <string>
#include <vector>
#ifdef _OPENMP
#include <omp.h>
#endif

namespace {

enum Precision { P_FP32 = 0, P_BF16 = 1, P_INT8 = 2 };

// ---- bf16 round-to-nearest-even, by bit manipulation (R20) -----------------
inline float bf16_round(float x) {
  uint32_t u;
  std::memcpy(&u, &x, 4);
  if ((u & 0x7f800000u) == 0x7f800000u) {          // inf / nan: truncate, keep nan a nan
    if (u & 0x007fffffu) u |= 0x00400000u;
    u &= 0xffff0000u;
  } else {
    uint32_t lsb = (u >> 16) & 1u;
    u += 0x7fffu + lsb;
    u &= 0xffff0000u;
  }
  float r;
  std::memcpy(&r, &u, 4);
  return r;
}

// ---- int8 symmetric quantiser (R21) -----------------------------------------
// q = clamp(rne(x * inv_s), -127, 127), inv_s = 1/s computed once in fp32.
inline int32_t quant_i8(float x, float inv_s) {
  float t = x * inv_s;                 // one fp32 multiply
  float r = std::nearbyintf(t);        // default rounding mode: to nearest even
  if (!(r >= -127.0f)) r = -127.0f;    // also catches NaN -> -127 (never occurs on finite inputs)
  if (r > 127.0f) r = 127.0f;
  return (int32_t)r;
}

struct Linear {
  int out = 0, in = 0;
  bool tensor = false;                  // in >= 16 and not the head  (R20/R21)
  std::vector<float> W, b;              // W[out][in] as in the blob
  std::vector<float> Wt;                // [in][out]: the weights the mode uses (fp32 or bf16-rounded)
  std::vector<int8_t> Wq;               // [out][in] (int8 mode, tensor layers)
  std::vector<float> sw;                // per-output-channel weight scale
  float sx = 1.0f, inv_sx = 1.0f;       // activation scale of this layer's input tensor
  int index = -1;                       // position in blob order
};

struct Model {
  int n_planes = 26;
  float norm_off[3] = {0, 0, 300}, norm_div[3] = {40, 40, 1050};
  int emb_input = 0;                    // 0: the embedding reads the Cartesian features; 1: cylindrical (L96, R27)
  float cyl_off[3] = {-20, 0, 300}, cyl_div[3] = {12, 3.14159274f, 1050};
  int emb_hidden = 0, emb_layers_hidden = 0, emb_dim = 4;
  int latent = 0, iters = 0, edge_enc_input = 0;
  int precision = P_FP32;
  int state_bf16 = 0;                   // h, e, m stored as bf16: always in bf16 mode; optional in int8 mode (R21)
  std::vector<Linear> emb;              // H+1 layers
  Linear nenc[2], eenc[2];
  std::vector<Linear> node, edge;       // 2 per iteration
  Linear head;
  int has_triplets = 0;                 // blob header word 11: the two triplet classifiers follow the head (L160)
  Linear tart[2], telb[2];              // articulation / elbow classifier: 2d -> d -> 1
  std::vector<Linear*> all;             // blob order
  std::string error;
  // instrumentation (not part of the method)
  std::vector<float> absmax;            // per layer: max |x| over inputs seen (calibration)
  bool record_absmax = false;
  int tap_layer = -1;                   // int8: copy this layer's int32 accumulators
  int32_t* tap_out = nullptr;           // [rows][out]
};

// y[c] = ( ... fmaf(x[1],W[c][1], fmaf(x[0],W[c][0], 0)) ... ) + b[c]      (R3, R4)
// Loop order j outer / c inner so the compiler can vectorise over output
// channels; each output's chain is still ascending j from 0.
inline void dense_f32(const Linear& L, const float* x, float* y) {
  float acc[256];
  const int O = L.out;
  for (int c = 0; c < O; ++c) acc[c] = 0.0f;
  for (int j = 0; j < L.in; ++j) {
    const float xj = x[j];
    const float* wt = &L.Wt[(size_t)j * O];
    for (int c = 0; c < O; ++c) acc[c] = std::fmaf(xj, wt[c], acc[c]);
  }
  for (int c = 0; c < O; ++c) y[c] = acc[c] + L.b[c];
}

// int8 x int8 -> int32, then y = fmaf((float)acc, sx*sw[c], b[c])            (R21)
inline void dense_i8(const Linear& L, const float* x, float* y, int32_t* acc_out) {
  int32_t q[256 * 3];
  for (int j = 0; j < L.in; ++j) q[j] = quant_i8(x[j], L.inv_sx);
  for (int c = 0; c < L.out; ++c) {
    int32_t acc = 0;
    const int8_t* w = &L.Wq[(size_t)c * L.in];
    for (int j = 0; j < L.in; ++j) acc += q[j] * (int32_t)w[j];
    if (acc_out) acc_out[c] = acc;
    const float scale = L.sx * L.sw[c];             // one fp32 product
    y[c] = std::fmaf((float)acc, scale, L.b[c]);
  }
}

// One Linear in the model's precision mode.  `row` only addresses the tap.
inline void linear(Model& M, const Linear& L, const float* x, float* y, size_t row) {
  if (M.record_absmax) {
    float m = 0.0f;
    for (int j = 0; j < L.in; ++j) m = std::max(m, std::fabs(x[j]));
    float& slot = M.absmax[L.index];
#pragma omp critical(etxo_absmax)
    { if (m > slot) slot = m; }
  }
  if (M.precision == P_INT8 && L.tensor) {
    int32_t* tap = (M.tap_layer == L.index && M.tap_out) ? M.tap_out + row * (size_t)L.out : nullptr;
    dense_i8(L, x, y, tap);
  } else {
    dense_f32(L, x, y);
  }
}

inline void relu(float* v, int n) { for (int i = 0; i < n; ++i) v[i] = v[i] > 0.0f ? v[i] : 0.0f; }
// Rounding points (R20).  operand_round: a hidden activation fed to a bf16 MMA (bf16 mode only; in int8 mode the
// operand is the int8 code, quantised from the fp32 value).  state_round: a stored state row h / e / m -- bf16 in
// bf16 mode, and in int8 mode when the state dtype is bf16 (R21: "if bf16 is adopted for bandwidth, mirror the RNE
// rounding in the oracle").
inline void operand_round(const Model& M, float* v, int n) {
  if (M.precision == P_BF16) for (int i = 0; i < n; ++i) v[i] = bf16_round(v[i]);
}
inline void state_round(const Model& M, float* v, int n) {
  if (M.state_bf16) for (int i = 0; i < n; ++i) v[i] = bf16_round(v[i]);
}

// f = ((x,y,z) + offset) / div : one fp32 add, one correctly rounded fp32 division (R1; L107 fn.5)
inline void features(const Model& M, const float* xyz, float* f) {
  for (int i = 0; i < 3; ++i) f[i] = (xyz[i] + M.norm_off[i]) / M.norm_div[i];
}

// Cylindrical embedding input (L96 "normalised cylindrical coordinates", R27).  r and phi in fp32, every step one
// correctly rounded operation in this order so that the CUDA path can take the same steps:
//   r   = sqrt(fma(y, y, x*x))
//   phi = atan2(y, x) through an odd polynomial on [0, 1]:  a = min(|x|,|y|) / max(|x|,|y|)  (0 if both are 0),
//         s = a*a,  q = Horner in s with fma over the nine coefficients below (degree 8, from c8 down to c0),
//         p = a*q;  |y| > |x|: p = pi/2 - p;  x < 0 (sign bit clear test on the value, so x = -0 counts as +0):
//         p = pi - p;  phi = copysign(p, y).
// |phi - atan2(y,x)| <= 5e-7 (pinned against the float64 library atan2); phi(0,0) = 0.
// The coefficients are a Chebyshev-node interpolant of atan(sqrt(s))/sqrt(s) on s in [0,1], rounded to fp32.
constexpr float kAtanC[9] = {0x1.000000p+0f,  -0x1.55548ep-2f, 0x1.996efcp-3f,  -0x1.22c55ap-3f, 0x1.b2edb0p-4f,
                             -0x1.316ecap-4f, 0x1.593100p-5f,  -0x1.01bda4p-6f, 0x1.6a9512p-9f};
inline float atan2_poly(float y, float x) {
  const float ax = std::fabs(x), ay = std::fabs(y);
  const float mx = ax > ay ? ax : ay, mn = ax > ay ? ay : ax;
  const float a = mx > 0.0f ? mn / mx : 0.0f;
  const float s = a * a;
  float q = kAtanC[8];
  for (int i = 7; i >= 0; --i) q = std::fmaf(q, s, kAtanC[i]);
  float p = a * q;
  if (ay > ax) p = 1.57079637f - p;
  if (x < 0.0f) p = 3.14159274f - p;
  return std::copysign(p, y);
}
// Input of the embedding MLP: the Cartesian features (emb_input 0, BASELINE configs, R1) or
// ((r, phi, z) + cyl_off) / cyl_div (emb_input 1, L96; same add-then-divide as R1).
inline void features_emb(const Model& M, const float* xyz, float* f) {
  if (!M.emb_input) { features(M, xyz, f); return; }
  const float x = xyz[0], y = xyz[1];
  const float c[3] = {std::sqrt(std::fmaf(y, y, x * x)), atan2_poly(y, x), xyz[2]};
  for (int i = 0; i < 3; ++i) f[i] = (c[i] + M.cyl_off[i]) / M.cyl_div[i];
}

bool parse_blob(Model& M, const uint8_t* blob, size_t bytes) {
  if (bytes < 64) { M.error = "blob too small"; return false; }
  uint32_t h[16];
  std::memcpy(h, blob, 64);
  if (h[0] != 0x57585445u || h[1] != 1u) { M.error = "bad magic/version"; return false; }
  M.emb_hidden = (int)h[2]; M.emb_layers_hidden = (int)h[3]; M.emb_dim = (int)h[4];
  M.latent = (int)h[5]; M.iters = (int)h[6]; M.edge_enc_input = (int)h[7];
  M.emb_input = (int)h[10];
  if (M.emb_input != 0 && M.emb_input != 1) { M.error = "bad emb_input"; return false; }
  M.has_triplets = (int)h[11];
  if (M.has_triplets != 0 && M.has_triplets != 1) { M.error = "bad triplet flag"; return false; }
  const int D = M.emb_hidden, H = M.emb_layers_hidden, d = M.latent, L = M.iters;
  if (D < 1 || D > 256 || H < 1 || H > 8 || M.emb_dim < 1 || M.emb_dim > 16 || d < 1 || d > 85 ||
      L < 0 || L > 64) { M.error = "bad shapes"; return false; }
  M.emb.resize(H + 1);
  M.node.resize(2 * L); M.edge.resize(2 * L);
  auto set = [&](Linear& l, int o, int i, bool head = false) {
    l.out = o; l.in = i; l.tensor = (i >= 16) && !head; M.all.push_back(&l);
  };
  set(M.emb[0], D, 3);
  for (int i = 1; i < H; ++i) set(M.emb[i], D, D);
  set(M.emb[H], M.emb_dim, D);
  set(M.nenc[0], d, 3); set(M.nenc[1], d, d);
  set(M.eenc[0], d, M.edge_enc_input ? 2 * d : 3); set(M.eenc[1], d, d);
  for (int it = 0; it < L; ++it) {
    set(M.node[2 * it], d, 3 * d); set(M.node[2 * it + 1], d, d);
    set(M.edge[2 * it], d, 3 * d); set(M.edge[2 * it + 1], d, d);
  }
  set(M.head, 1, d, true);
  if (M.has_triplets) {                 // L160: "an MLP ending with a layer with 1 unit" for articulations, one for elbows (R28)
    set(M.tart[0], d, 2 * d); set(M.tart[1], 1, d, true);
    set(M.telb[0], d, 2 * d); set(M.telb[1], 1, d, true);
  }
  size_t need = 0; int nq = 0;
  for (Linear* l : M.all) { need += (size_t)l->out * l->in + l->out; nq += l->tensor; }
  if (h[8] != need) { M.error = "n_weight_floats mismatch"; return false; }
  const size_t n_scales = h[9];
  if (bytes != 64 + 4 * (need + n_scales)) { M.error = "blob size mismatch"; return false; }
  if (M.precision == P_INT8 && (int)n_scales != nq) { M.error = "int8 needs one act scale per quantised layer"; return false; }
  const float* p = reinterpret_cast<const float*>(blob + 64);
  const float* scales = p + need;
  int idx = 0, qi = 0;
  for (Linear* l : M.all) {
    l->index = idx++;
    l->W.assign(p, p + (size_t)l->out * l->in); p += (size_t)l->out * l->in;
    l->b.assign(p, p + l->out); p += l->out;
    const bool round_w = (M.precision == P_BF16 && l->tensor);
    l->Wt.resize((size_t)l->in * l->out);
    for (int c = 0; c < l->out; ++c)
      for (int j = 0; j < l->in; ++j) {
        float w = l->W[(size_t)c * l->in + j];
        l->Wt[(size_t)j * l->out + c] = round_w ? bf16_round(w) : w;
      }
    if (M.precision == P_INT8 && l->tensor) {
      // per-output-channel symmetric weight scale s_w = max|w|/127 (1 if the row is zero)  (R21)
      l->sw.resize(l->out); l->Wq.resize((size_t)l->out * l->in);
      for (int c = 0; c < l->out; ++c) {
        float m = 0.0f;
        for (int j = 0; j < l->in; ++j) m = std::max(m, std::fabs(l->W[(size_t)c * l->in + j]));
        float s = (m > 0.0f) ? m / 127.0f : 1.0f;
        l->sw[c] = s;
        for (int j = 0; j < l->in; ++j) {
          float t = l->W[(size_t)c * l->in + j] / s;           // correctly rounded division
          float r = std::nearbyintf(t);
          r = std::min(127.0f, std::max(-127.0f, r));
          l->Wq[(size_t)c * l->in + j] = (int8_t)r;
        }
      }
      l->sx = scales[qi++];
      if (!(l->sx > 0.0f)) { M.error = "activation scale must be > 0"; return false; }
      l->inv_sx = 1.0f / l->sx;
    }
  }
  M.absmax.assign(M.all.size(), 0.0f);
  return true;
}

}  // namespace

// ============================================================================
extern "C" {

struct etxo_params {
  int32_t n_planes;
  float norm_offset[3];
  float norm_div[3];
  int32_t precision;   // 0 fp32, 1 bf16-emulated, 2 int8
  float cyl_offset[3]; // used when the blob says emb_input = 1 (R27)
  float cyl_div[3];
  int32_t state_dtype; // 0: fp32 for fp32 / int8, bf16 for bf16 (the defaults); 1: fp32; 2: bf16 (int8 mode only)
};

void* etxo_create(const void* blob, uint64_t bytes, const etxo_params* prm) {
  Model* M = new Model();
  M->precision = prm->precision;
  M->state_bf16 = (prm->precision == P_BF16) || (prm->precision == P_INT8 && prm->state_dtype == 2);
  M->n_planes = prm->n_planes;
  for (int i = 0; i < 3; ++i) { M->norm_off[i] = prm->norm_offset[i]; M->norm_div[i] = prm->norm_div[i]; }
  for (int i = 0; i < 3; ++i) { M->cyl_off[i] = prm->cyl_offset[i]; M->cyl_div[i] = prm->cyl_div[i]; }
  if (!parse_blob(*M, static_cast<const uint8_t*>(blob), (size_t)bytes)) { /* keep M for the message */ }
  return M;
}
const char* etxo_error(void* m) { return static_cast<Model*>(m)->error.c_str(); }
void etxo_destroy(void* m) { delete static_cast<Model*>(m); }
int etxo_threads() {
#ifdef _OPENMP
  return omp_get_max_threads();
#else
  return 1;
#endif
}
void etxo_set_threads(int n) {
#ifdef _OPENMP
  omp_set_num_threads(n);
#else
  (void)n;
#endif
}

float etxo_bf16_round(float x) { return bf16_round(x); }
int32_t etxo_quant_i8(float x, float scale) { return quant_i8(x, 1.0f / scale); }

// instrumentation controls
void etxo_record_absmax(void* m, int on) {
  Model* M = static_cast<Model*>(m);
  M->record_absmax = on != 0;
  if (on) std::fill(M->absmax.begin(), M->absmax.end(), 0.0f);
}
int etxo_n_layers(void* m) { return (int)static_cast<Model*>(m)->all.size(); }
void etxo_get_absmax(void* m, float* out) {
  Model* M = static_cast<Model*>(m);
  std::copy(M->absmax.begin(), M->absmax.end(), out);
}
// s_x = max|x| / 127 (1 if zero), for the quantised layers in blob order (R21).  Returns count.
int etxo_scales_from_absmax(void* m, float* out) {
  Model* M = static_cast<Model*>(m);
  int n = 0;
  for (Linear* l : M->all)
    if (l->tensor) { float a = M->absmax[l->index]; out[n++] = (a > 0.0f) ? a / 127.0f : 1.0f; }
  return n;
}
void etxo_set_tap(void* m, int layer_index, int32_t* out) {
  Model* M = static_cast<Model*>(m);
  M->tap_layer = layer_index; M->tap_out = out;
}
// quantised weights of one layer (for the integer-matmul pin); returns 0 if not quantised
int etxo_get_qweights(void* m, int layer_index, int8_t* Wq, float* sw, float* sx) {
  Model* M = static_cast<Model*>(m);
  Linear* l = M->all[layer_index];
  if (l->Wq.empty()) return 0;
  std::copy(l->Wq.begin(), l->Wq.end(), Wq);
  std::copy(l->sw.begin(), l->sw.end(), sw);
  *sx = l->sx;
  return 1;
}

// ---------------------------------------------------------------------------
// Step 0.  Plane offsets: plane_off[e*(P+1)+p] = first hit (global index) of
// event e whose plane is >= p; entry P is the event's end.  Hits arrive
// sorted by (event, plane) (Allen decodes hits per module).
void etxo_plane_offsets(const int32_t* plane, const int32_t* event_off, int n_events, int P, int32_t* plane_off) {
  for (int e = 0; e < n_events; ++e) {
    int32_t i = event_off[e];
    const int32_t end = event_off[e + 1];
    for (int p = 0; p <= P; ++p) {
      while (i < end && plane[i] < p) ++i;
      plane_off[(size_t)e * (P + 1) + p] = i;
    }
  }
}

// Step 1 (normalisation only; exported for the pins).
void etxo_features(void* m, const float* xyz, int64_t n, float* f) {
  Model& M = *static_cast<Model*>(m);
  for (int64_t i = 0; i < n; ++i) features(M, xyz + 3 * i, f + 3 * i);
}

void etxo_features_emb(void* m, const float* xyz, int64_t n, float* f) {
  const Model& M = *static_cast<Model*>(m);
  for (int64_t i = 0; i < n; ++i) features_emb(M, xyz + 3 * i, f + 3 * i);
}

// ---------------------------------------------------------------------------
// Step 1+2.  Hit embedding (section 5.1): e_h = MLP(normalised coords);
// ReLU after hidden layers, linear output (R3).  bf16 mode rounds every hidden
// activation (they feed the next MMA) but not the fp32 output (R20).
void etxo_embed(void* m, const float* xyz, int64_t n, float* emb) {
  Model& M = *static_cast<Model*>(m);
  const int H = M.emb_layers_hidden;
#pragma omp parallel for schedule(static)
  for (int64_t i = 0; i < n; ++i) {
    float a[256], t[256], f[3];
    features_emb(M, xyz + 3 * i, f);
    linear(M, M.emb[0], f, a, (size_t)i);
    relu(a, M.emb[0].out); operand_round(M, a, M.emb[0].out);
    for (int l = 1; l < H; ++l) {
      linear(M, M.emb[l], a, t, (size_t)i);
      relu(t, M.emb[l].out); operand_round(M, t, M.emb[l].out);
      std::memcpy(a, t, sizeof(float) * M.emb[l].out);
    }
    linear(M, M.emb[H], a, emb + (size_t)i * M.emb_dim, (size_t)i);
  }
}

// ---------------------------------------------------------------------------
// Step 3.  Plane-restricted k-NN (Eq.(1), L101, L257 section 7.2).
// For hit q on plane p the candidates are the hits of the same event on planes
// p+1 .. min(p+w, P-1): a contiguous index range.  d2 is Eq.(1) evaluated as
// t0*t0, then fmaf(t_i, t_i, d2) for i = 1.. (R4).  Candidates with d2 < d2_max
// (strict, R6) are kept; the result is the first min(k, kept) of them in
// ascending (d2, index) order (R5).  This is the paper's sequential scan with a
// k-slot list (L257), the list kept sorted so that ties resolve to the lower
// hit index.  nbr is [n][k], -1 padded; deg[n].
void etxo_knn(const float* emb, int64_t n, int n_dim, const int32_t* plane, const int32_t* event_off,
              int n_events, int P, int k, int w, float d2_max, int32_t* nbr, int32_t* deg) {
  std::vector<int32_t> plane_off((size_t)n_events * (P + 1));
  etxo_plane_offsets(plane, event_off, n_events, P, plane_off.data());
  for (int e = 0; e < n_events; ++e) {
    const int32_t* po = &plane_off[(size_t)e * (P + 1)];
#pragma omp parallel for schedule(dynamic, 16)
    for (int32_t q = event_off[e]; q < event_off[e + 1]; ++q) {
      const int p = plane[q];
      const int p_hi = std::min(p + w, P - 1);
      std::vector<float> ld(k);          // list, ascending (d2, index)
      std::vector<int32_t> li(k);
      int cnt = 0;
      if (p + 1 <= p_hi) {
        for (int32_t c = po[p + 1]; c < po[p_hi + 1]; ++c) {
          const float* a = emb + (size_t)q * n_dim;
          const float* b = emb + (size_t)c * n_dim;
          float t = a[0] - b[0];
          float d2 = t * t;
          for (int i = 1; i < n_dim; ++i) { t = a[i] - b[i]; d2 = std::fmaf(t, t, d2); }
          if (!(d2 < d2_max)) continue;
          // candidates arrive in ascending index, so an equal d2 goes after the ones present
          int pos = cnt;
          while (pos > 0 && d2 < ld[pos - 1]) --pos;
          if (pos >= k) continue;
          const int last = std::min(cnt, k - 1);
          for (int s = last; s > pos; --s) { ld[s] = ld[s - 1]; li[s] = li[s - 1]; }
          ld[pos] = d2; li[pos] = c;
          if (cnt < k) ++cnt;
        }
      }
      deg[q] = cnt;
      for (int s = 0; s < k; ++s) nbr[(size_t)q * k + s] = s < cnt ? li[s] : -1;
    }
  }
}

// Step 4.  Edge list G_rough (directed i -> j, i on the
// lower plane): concatenation over q ascending of q's neighbours in rank order (R9).
// row_ptr[n+1] = prefix sums of deg.  Returns E.
int64_t etxo_build_edges(const int32_t* nbr, const int32_t* deg, int64_t n, int k,
                         int32_t* src, int32_t* dst, int32_t* row_ptr) {
  int64_t E = 0;
  for (int64_t q = 0; q < n; ++q) {
    row_ptr[q] = (int32_t)E;
    for (int s = 0; s < deg[q]; ++s) { src[E] = (int32_t)q; dst[E] = nbr[q * k + s]; ++E; }
  }
  row_ptr[n] = (int32_t)E;
  return E;
}

// In-edge lists: in_edge grouped by dst, ascending edge id inside a group; col_ptr[n+1].
void etxo_csc(const int32_t* dst, int64_t E, int64_t n, int32_t* col_ptr, int32_t* in_edge) {
  std::vector<int32_t> cnt(n + 1, 0);
  for (int64_t i = 0; i < E; ++i) cnt[dst[i] + 1]++;
  col_ptr[0] = 0;
  for (int64_t l = 0; l < n; ++l) col_ptr[l + 1] = col_ptr[l] + cnt[l + 1];
  std::vector<int32_t> cur(col_ptr, col_ptr + n);
  for (int64_t i = 0; i < E; ++i) in_edge[cur[dst[i]]++] = (int32_t)i;
}

// ---------------------------------------------------------------------------
// Step 5-7.  Interaction-network edge classifier (section 5.2).
//   h0 = MLP_ne(f)                                        node encoder (L133)
//   e0 = MLP_ee(|f_dst - f_src|)   or MLP_ee([h0_src,h0_dst]) (R10: configs vs L133)
//   for k = 0..L-1                                        (L135-140, distinct weights L148)
//     m_out[l] = sum_{l->j} e_lj ; m_in[l] = sum_{i->l} e_il   (Eq.(4)), fp32, ascending edge id (R22)
//     h <- h + MLP_k^node([h, m_out, m_in])                 residual (L140, R14)
//     e <- e + MLP_k^edge([h_src, h_dst, e])  with the UPDATED h (L140, R13)
//   z = w_head . e + b ; score = sigmoid(z)                (L80, L142, R16)
// Outputs: logit[E], score[E]; optional h_out[n][d], e_out[E][d] (final states);
// optional m_out_dump[n][2d] = the message of iteration `m_iter`.
void etxo_gnn(void* m, const float* xyz, int64_t n, const int32_t* src, const int32_t* dst, int64_t E,
              float* logit, float* score, float* h_out, float* e_out, float* m_dump, int m_iter) {
  Model& M = *static_cast<Model*>(m);
  const int d = M.latent;
  std::vector<float> f((size_t)n * 3), h((size_t)n * d), e((size_t)E * d), msg((size_t)n * 2 * d);
  for (int64_t i = 0; i < n; ++i) features(M, xyz + 3 * i, &f[3 * i]);

#pragma omp parallel for schedule(static)
  for (int64_t i = 0; i < n; ++i) {                       // node encoder
    float a[96], t[96];
    linear(M, M.nenc[0], &f[3 * i], a, (size_t)i);
    relu(a, d); operand_round(M, a, d);
    linear(M, M.nenc[1], a, t, (size_t)i);
    state_round(M, t, d);
    std::memcpy(&h[(size_t)i * d], t, sizeof(float) * d);
  }
#pragma omp parallel for schedule(static)
  for (int64_t i = 0; i < E; ++i) {                       // edge encoder
    float x[192], a[96], t[96];
    if (M.edge_enc_input == 0) {
      for (int c = 0; c < 3; ++c) x[c] = std::fabs(f[3 * (size_t)dst[i] + c] - f[3 * (size_t)src[i] + c]);  // R11
    } else {
      std::memcpy(x, &h[(size_t)src[i] * d], sizeof(float) * d);
      std::memcpy(x + d, &h[(size_t)dst[i] * d], sizeof(float) * d);
    }
    linear(M, M.eenc[0], x, a, (size_t)i);
    relu(a, d); operand_round(M, a, d);
    linear(M, M.eenc[1], a, t, (size_t)i);
    state_round(M, t, d);
    std::memcpy(&e[(size_t)i * d], t, sizeof(float) * d);
  }

  for (int it = 0; it < M.iters; ++it) {
    // message building, Eq.(4): one loop over edges in ascending edge id (R22)
    std::fill(msg.begin(), msg.end(), 0.0f);
    for (int64_t i = 0; i < E; ++i) {
      float* mo = &msg[(size_t)src[i] * 2 * d];
      float* mi = &msg[(size_t)dst[i] * 2 * d + d];
      const float* ee = &e[(size_t)i * d];
      for (int c = 0; c < d; ++c) { mo[c] += ee[c]; mi[c] += ee[c]; }
    }
    // bf16 state: the message is stored (and is a tensor-core operand), rounded once after the fp32 sum (R20)
    if (M.state_bf16) for (size_t i = 0; i < msg.size(); ++i) msg[i] = bf16_round(msg[i]);
    if (m_dump && it == m_iter) std::memcpy(m_dump, msg.data(), sizeof(float) * msg.size());

#pragma omp parallel for schedule(static)
    for (int64_t i = 0; i < n; ++i) {                     // node network
      float x[288], a[96], t[96];
      std::memcpy(x, &h[(size_t)i * d], sizeof(float) * d);
      std::memcpy(x + d, &msg[(size_t)i * 2 * d], sizeof(float) * 2 * d);
      linear(M, M.node[2 * it], x, a, (size_t)i);
      relu(a, d); operand_round(M, a, d);
      linear(M, M.node[2 * it + 1], a, t, (size_t)i);
      float* hh = &h[(size_t)i * d];
      for (int c = 0; c < d; ++c) hh[c] = hh[c] + t[c];   // residual, fp32 add (R14)
      state_round(M, hh, d);
    }
#pragma omp parallel for schedule(static)
    for (int64_t i = 0; i < E; ++i) {                     // edge network (uses the updated h)
      float x[288], a[96], t[96];
      std::memcpy(x, &h[(size_t)src[i] * d], sizeof(float) * d);
      std::memcpy(x + d, &h[(size_t)dst[i] * d], sizeof(float) * d);
      std::memcpy(x + 2 * d, &e[(size_t)i * d], sizeof(float) * d);
      linear(M, M.edge[2 * it], x, a, (size_t)i);
      relu(a, d); operand_round(M, a, d);
      linear(M, M.edge[2 * it + 1], a, t, (size_t)i);
      float* ee = &e[(size_t)i * d];
      for (int c = 0; c < d; ++c) ee[c] = ee[c] + t[c];
      state_round(M, ee, d);
    }
  }
#pragma omp parallel for schedule(static)
  for (int64_t i = 0; i < E; ++i) {                       // edge classifier head (R16)
    float z;
    linear(M, M.head, &e[(size_t)i * d], &z, (size_t)i);
    logit[i] = z;
    score[i] = (float)(1.0 / (1.0 + std::exp(-(double)z)));
  }
  if (h_out) std::memcpy(h_out, h.data(), sizeof(float) * h.size());
  if (e_out) std::memcpy(e_out, e.data(), sizeof(float) * e.size());
}

// tau = (float) log(thr / (1 - thr)) ; an edge is kept iff logit >= tau (L80 "below ... discarded", R17)
float etxo_logit_threshold(float thr) {
  if (thr <= 0.0f) return -std::numeric_limits<float>::infinity();
  if (thr >= 1.0f) return std::numeric_limits<float>::infinity();
  return (float)std::log((double)thr / (1.0 - (double)thr));
}

// ---------------------------------------------------------------------------
// Step 8-9.  Threshold + weakly connected components of the purified hit graph
// (section 7.3).  track_id[h] = smallest global hit index
// in h's component ("each node is initially assigned ... its own node index",
// the lowest label propagates; R18: exact components instead of two sweeps).
// Sequential union-find, root = smaller index, then one pass of find.
void etxo_components(const int32_t* src, const int32_t* dst, const float* logit, int64_t E, float tau,
                     int64_t n, int32_t* track_id) {
  std::vector<int32_t> parent(n);
  for (int64_t i = 0; i < n; ++i) parent[i] = (int32_t)i;
  auto find = [&](int32_t x) {
    while (parent[x] != x) { parent[x] = parent[parent[x]]; x = parent[x]; }
    return x;
  };
  for (int64_t i = 0; i < E; ++i) {
    if (!(logit[i] >= tau)) continue;
    int32_t a = find(src[i]), b = find(dst[i]);
    if (a == b) continue;
    if (a < b) parent[b] = a; else parent[a] = b;
  }
  for (int64_t i = 0; i < n; ++i) track_id[i] = find((int32_t)i);
}

// ---------------------------------------------------------------------------
// Track containers (a particle is reconstructible in the VELO with at
// least three hits; L74, L82: the output of the pipeline is the set of tracks, each a list of hits).  A track is
// a connected component with at least min_hits hits.  Tracks are numbered densely in ascending order of their
// smallest hit index (= their track_id), so the tracks of one event are consecutive; hits inside a track are in
// ascending hit index.  Outputs:
//   track_index[n]        dense track number of the hit's track, or -1 (component too small)
//   track_offsets[T + 1]  CSR offsets into track_hits            (capacity n + 1)
//   track_hits[...]       hit indices, track after track          (capacity n)
//   event_track_off[B+1]  first dense track number of every event
// Returns T.  Plain loops: count, number, fill.
int64_t etxo_tracks(const int32_t* track_id, int64_t n, const int32_t* event_off, int64_t n_events, int32_t min_hits,
                    int32_t* track_index, int32_t* track_offsets, int32_t* track_hits, int32_t* event_track_off) {
  std::vector<int32_t> size(n, 0), number(n, -1);
  for (int64_t h = 0; h < n; ++h) size[track_id[h]] += 1;             // component size, stored at its root
  int64_t T = 0;
  track_offsets[0] = 0;
  for (int64_t r = 0; r < n; ++r) {                                   // roots in ascending order
    if (track_id[r] == r && size[r] >= min_hits) {
      number[r] = (int32_t)T;
      track_offsets[T + 1] = track_offsets[T] + size[r];
      ++T;
    }
  }
  std::vector<int32_t> cursor(track_offsets, track_offsets + T);
  for (int64_t h = 0; h < n; ++h) {                                   // hits in ascending order -> ascending inside a track
    const int32_t t = number[track_id[h]];
    track_index[h] = t;
    if (t >= 0) track_hits[cursor[t]++] = (int32_t)h;
  }
  for (int64_t e = 0; e <= n_events; ++e) {                           // tracks whose root lies before the event's first hit
    int64_t cnt = 0;
    const int64_t lim = e < n_events ? event_off[e] : n;
    for (int64_t r = 0; r < lim; ++r) cnt += number[r] >= 0;
    event_track_off[e] = (int32_t)cnt;
  }
  return T;
}

// ---------------------------------------------------------------------------
// Triplet stage (sec. 5.3, sec. 5.4).  The paper left it out of
// its CUDA code (L238); readings R28-R31 in DESIGN.md say what is built where the text is silent.
//
// Triplet building (L152-158) on the purified hit graph (edges with keep[i] != 0, i.e. logit >= tau, L80 / L146).
// A triplet is a pair of kept edges (first, second) with one common hit C:
//   kind 0  articulation  A -> C, C -> B : first = the in-edge of C, second = the out-edge of C
//   kind 1  left elbow    C -> A, C -> B : two distinct out-edges of C, first < second (edge id)
//   kind 2  right elbow   A -> C, B -> C : two distinct in-edges of C,  first < second (edge id)
// Order (R29): common hit C ascending, then first ascending, then second ascending.  Returns the number of
// triplets; t_first / t_second / t_hit (each may be null: count only) receive the edge ids and the common hit.
int64_t etxo_triplets(const int32_t* src, const int32_t* dst, const uint8_t* keep, int64_t E, int64_t n, int kind,
                      int32_t* t_first, int32_t* t_second, int32_t* t_hit) {
  std::vector<std::vector<int32_t>> out(n), in(n);               // kept edges per hit, ascending edge id
  for (int64_t i = 0; i < E; ++i)
    if (keep[i]) { out[src[i]].push_back((int32_t)i); in[dst[i]].push_back((int32_t)i); }
  int64_t T = 0;
  auto emit = [&](int32_t a, int32_t b, int64_t c) {
    if (t_first) t_first[T] = a;
    if (t_second) t_second[T] = b;
    if (t_hit) t_hit[T] = (int32_t)c;
    ++T;
  };
  for (int64_t c = 0; c < n; ++c) {
    if (kind == 0) {
      for (int32_t a : in[c]) for (int32_t b : out[c]) emit(a, b, c);
    } else {
      const std::vector<int32_t>& l = kind == 1 ? out[c] : in[c];
      for (size_t i = 0; i < l.size(); ++i) for (size_t j = i + 1; j < l.size(); ++j) emit(l[i], l[j], c);
    }
  }
  return T;
}

// Triplet classifier (L80: "transforms the pairs of edge encodings (triplets) into triplet scores"; L160: separate
// classifiers for articulations and elbows, each "an MLP ending with a layer with 1 unit, and a sigmoid").
// R28: input [e_first, e_second] (2d) of the FINAL edge encodings e^L, one hidden layer of width d with ReLU, then
// d -> 1; z = logit, score = sigmoid(z).  `elbow` selects the classifier.  Precision modes as everywhere else
// (R20 / R21): the 2d -> d layer is a tensor layer (bf16 weights / int8 codes, hidden activation rounded in bf16
// mode), the d -> 1 layer is fp32 in the pinned order like the edge head.
void etxo_triplet_scores(void* m, const float* e_state, const int32_t* t_first, const int32_t* t_second, int64_t T,
                         int elbow, float* logit, float* score) {
  Model& M = *static_cast<Model*>(m);
  const int d = M.latent;
  Linear* L = elbow ? M.telb : M.tart;
#pragma omp parallel for schedule(static)
  for (int64_t t = 0; t < T; ++t) {
    float x[192], a[96], z;
    std::memcpy(x, e_state + (size_t)t_first[t] * d, sizeof(float) * d);
    std::memcpy(x + d, e_state + (size_t)t_second[t] * d, sizeof(float) * d);
    linear(M, L[0], x, a, (size_t)t);
    relu(a, d); operand_round(M, a, d);
    linear(M, L[1], a, &z, (size_t)t);
    logit[t] = z;
    score[t] = (float)(1.0 / (1.0 + std::exp(-(double)z)));
  }
}
int etxo_has_triplets(void* m) { return static_cast<Model*>(m)->has_triplets; }

// Track building from triplets (sec. 5.4, Figure 6), the four phases as read in R30:
//  (1) "the left elbows and right elbows are connected": the two edges of every kept elbow are merged into one
//      super-edge (union-find over edge ids, root = smallest id).  Articulations are mapped onto super-edges;
//      "duplicate edges resulting from elbow connections are removed": equal (first, second) pairs collapse, and an
//      articulation inside one super-edge disappears.
//  (2) An articulation is SHARED when its first super-edge has two or more distinct successors or its second one
//      two or more distinct predecessors ("two articulations sharing an edge").  WCC over the super-edges with the
//      non-shared articulations only.
//  (3) "a new track is formed for each remaining articulation, effectively duplicating the shared set": every shared
//      articulation (X, Y) yields the track comp(X) u comp(Y); a component touched by no shared articulation is a
//      track by itself.
//  (4) edges -> hits: a track's hits are the end points of its edges, ascending.  Tracks with fewer than min_hits
//      hits are dropped (L42), identical hit lists are kept once, and the result is ordered lexicographically by
//      hit list (R31), so that it can be compared as arrays.
// Only kept edges take part (an edge below the edge threshold is in no triplet, L146); a kept edge without any
// kept triplet is a component of its own (two hits).  keepA / keepL / keepR flag the kept triplets of each kind.
//
// The work is split in two so that the first half can be compared with the CUDA path, which stops there:
//   etxo_triplet_components  phases (1)-(2): edge_comp[e] = the component of kept edge e, named by the smallest edge
//                            id in it (-1 for an edge that is not kept), and the shared articulations as pairs of
//                            component names, sorted and without repeats (a pair with equal names is kept: it still
//                            marks its component as part of a shared structure).  Returns the number of pairs
//                            (capacity TA).
//   etxo_tracks_from_components  phases (3)-(4).
int64_t etxo_triplet_components(const uint8_t* keep, int64_t E,
                                const int32_t* a_first, const int32_t* a_second, const uint8_t* keepA, int64_t TA,
                                const int32_t* l_first, const int32_t* l_second, const uint8_t* keepL, int64_t TL,
                                const int32_t* r_first, const int32_t* r_second, const uint8_t* keepR, int64_t TR,
                                int32_t* edge_comp, int32_t* shared_x, int32_t* shared_y) {
  std::vector<int32_t> sup(E);
  for (int64_t i = 0; i < E; ++i) sup[i] = (int32_t)i;
  auto find = [](std::vector<int32_t>& p, int32_t x) {
    while (p[x] != x) { p[x] = p[p[x]]; x = p[x]; }
    return x;
  };
  auto unite = [&](std::vector<int32_t>& p, int32_t a, int32_t b) {
    a = find(p, a); b = find(p, b);
    if (a == b) return;
    if (a < b) p[b] = a; else p[a] = b;
  };
  // (1) elbows merge edges
  for (int64_t t = 0; t < TL; ++t) if (keepL[t]) unite(sup, l_first[t], l_second[t]);
  for (int64_t t = 0; t < TR; ++t) if (keepR[t]) unite(sup, r_first[t], r_second[t]);
  std::vector<std::pair<int32_t, int32_t>> arts;
  for (int64_t t = 0; t < TA; ++t)
    if (keepA[t]) {
      const int32_t x = find(sup, a_first[t]), y = find(sup, a_second[t]);
      if (x != y) arts.push_back({x, y});
    }
  std::sort(arts.begin(), arts.end());
  arts.erase(std::unique(arts.begin(), arts.end()), arts.end());
  // (2) shared articulations, WCC over the rest
  std::vector<int32_t> n_succ(E, 0), n_pred(E, 0);
  for (auto& a : arts) { n_succ[a.first]++; n_pred[a.second]++; }      // arts are distinct pairs
  std::vector<int32_t> comp(E);
  for (int64_t i = 0; i < E; ++i) comp[i] = (int32_t)i;
  std::vector<std::pair<int32_t, int32_t>> shared;
  for (auto& a : arts) {
    if (n_succ[a.first] >= 2 || n_pred[a.second] >= 2) shared.push_back(a);
    else unite(comp, a.first, a.second);
  }
  for (int64_t i = 0; i < E; ++i) edge_comp[i] = keep[i] ? find(comp, find(sup, (int32_t)i)) : -1;
  for (auto& a : shared) { a.first = find(comp, a.first); a.second = find(comp, a.second); }
  std::sort(shared.begin(), shared.end());
  shared.erase(std::unique(shared.begin(), shared.end()), shared.end());
  for (size_t i = 0; i < shared.size(); ++i) { shared_x[i] = shared[i].first; shared_y[i] = shared[i].second; }
  return (int64_t)shared.size();
}

// Outputs: track_offsets[T + 1], track_hits[...] (capacities given by the caller: cap_tracks + 1, cap_hits);
// returns T, or -1 if a capacity is too small.
int64_t etxo_tracks_from_components(const int32_t* src, const int32_t* dst, const int32_t* edge_comp, int64_t E,
                                    const int32_t* shared_x, const int32_t* shared_y, int64_t n_shared,
                                    int32_t min_hits, int32_t* track_offsets, int64_t cap_tracks,
                                    int32_t* track_hits, int64_t cap_hits) {
  // (3) tracks as sets of components
  std::vector<uint8_t> touched(E, 0);
  std::vector<std::vector<int32_t>> track_comps;
  for (int64_t i = 0; i < n_shared; ++i) {
    const int32_t p = shared_x[i], q = shared_y[i];
    touched[p] = touched[q] = 1;
    if (p == q) track_comps.push_back({p}); else track_comps.push_back({p, q});
  }
  std::vector<std::vector<int32_t>> members(E);                       // kept edges by component name
  for (int64_t i = 0; i < E; ++i) if (edge_comp[i] >= 0) members[edge_comp[i]].push_back((int32_t)i);
  for (int64_t i = 0; i < E; ++i) if (!members[i].empty() && !touched[i]) track_comps.push_back({(int32_t)i});
  // (4) edges -> hits
  std::vector<std::vector<int32_t>> tracks;
  for (auto& tc : track_comps) {
    std::vector<int32_t> hits;
    for (int32_t c : tc) for (int32_t e : members[c]) { hits.push_back(src[e]); hits.push_back(dst[e]); }
    std::sort(hits.begin(), hits.end());
    hits.erase(std::unique(hits.begin(), hits.end()), hits.end());
    if ((int32_t)hits.size() >= min_hits) tracks.push_back(hits);
  }
  std::sort(tracks.begin(), tracks.end());
  tracks.erase(std::unique(tracks.begin(), tracks.end()), tracks.end());
  if ((int64_t)tracks.size() > cap_tracks) return -1;
  int64_t pos = 0;
  track_offsets[0] = 0;
  for (size_t t = 0; t < tracks.size(); ++t) {
    if (pos + (int64_t)tracks[t].size() > cap_hits) return -1;
    for (int32_t h : tracks[t]) track_hits[pos++] = h;
    track_offsets[t + 1] = (int32_t)pos;
  }
  return (int64_t)tracks.size();
}

int64_t etxo_tracks_from_triplets(const int32_t* src, const int32_t* dst, const uint8_t* keep, int64_t E,
                                  const int32_t* a_first, const int32_t* a_second, const uint8_t* keepA, int64_t TA,
                                  const int32_t* l_first, const int32_t* l_second, const uint8_t* keepL, int64_t TL,
                                  const int32_t* r_first, const int32_t* r_second, const uint8_t* keepR, int64_t TR,
                                  int32_t min_hits, int32_t* track_offsets, int64_t cap_tracks,
                                  int32_t* track_hits, int64_t cap_hits) {
  std::vector<int32_t> edge_comp(E > 0 ? E : 1), sx(TA > 0 ? TA : 1), sy(TA > 0 ? TA : 1);
  const int64_t ns = etxo_triplet_components(keep, E, a_first, a_second, keepA, TA, l_first, l_second, keepL, TL,
                                             r_first, r_second, keepR, TR, edge_comp.data(), sx.data(), sy.data());
  return etxo_tracks_from_components(src, dst, edge_comp.data(), E, sx.data(), sy.data(), ns, min_hits,
                                     track_offsets, cap_tracks, track_hits, cap_hits);
}

}  // extern "C"
