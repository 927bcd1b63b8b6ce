// FFMA ("SIMT") kernels of the MLP stages S1 and S4 and the Eq.(4) scatter-sum.
//
// These run the fp32 precision mode (configs 0 and 1), and in every precision they are the deterministic
// debugging path (etx_engine = ETX_ENGINE_SIMT): each output is ONE sequential chain
//     acc = 0; for j ascending: acc = fmaf(x_j, w_j, acc);  y = fmaf(acc, scale, b)
// (scale = 1 outside INT8, where it is s_x*s_w[c]; R3/R4/R21), so results do not depend on the
// tiling.  INT8 is emulated exactly on the FFMA pipe: int8 codes are small integers, every partial sum is an
// integer below 2^24, so the fp32 chain reproduces the int32 accumulator bit for bit.
#include "etx_internal.h"

namespace etx {

enum { kModeF32 = 0, kModeBf16 = 1, kModeInt8 = 2 };

__device__ __forceinline__ float bf16r(float x) { return __bfloat162float(__float2bfloat16_rn(x)); }

// q = clamp(rne(x * inv_s), -127, 127) as a float (R21)
__device__ __forceinline__ float quant_i8(float x, float inv_s) {
  float r = rintf(__fmul_rn(x, inv_s));
  r = fmaxf(r, -127.0f);
  return fminf(r, 127.0f);
}

// ---- state access: fp32 or bf16 rows of d values, 4 at a time ---------------------------------------------
template <typename ST> struct State;
template <> struct State<float> {
  static __device__ __forceinline__ float4 ld4(const void* base, size_t elem) {
    return *reinterpret_cast<const float4*>(static_cast<const float*>(base) + elem);
  }
  static __device__ __forceinline__ void st4(void* base, size_t elem, float4 v) {
    *reinterpret_cast<float4*>(static_cast<float*>(base) + elem) = v;
  }
  static __device__ __forceinline__ float round(float x) { return x; }
};
template <> struct State<__nv_bfloat16> {
  static __device__ __forceinline__ float4 ld4(const void* base, size_t elem) {
    uint2 u = *reinterpret_cast<const uint2*>(static_cast<const __nv_bfloat16*>(base) + elem);
    return make_float4(__uint_as_float(u.x << 16), __uint_as_float(u.x & 0xffff0000u),
                       __uint_as_float(u.y << 16), __uint_as_float(u.y & 0xffff0000u));
  }
  static __device__ __forceinline__ void st4(void* base, size_t elem, float4 v) {   // values already rounded
    uint2 u;
    u.x = (__float_as_uint(v.x) >> 16) | (__float_as_uint(v.y) & 0xffff0000u);
    u.y = (__float_as_uint(v.z) >> 16) | (__float_as_uint(v.w) & 0xffff0000u);
    *reinterpret_cast<uint2*>(static_cast<__nv_bfloat16*>(base) + elem) = u;
  }
  static __device__ __forceinline__ float round(float x) { return bf16r(x); }
};

// hidden activation -> operand of the next (tensor) layer: bf16 rounding / int8 quantisation (R20, R21)
template <int MODE>
__device__ __forceinline__ float to_operand(float v, float inv_sx_next) {
  if (MODE == kModeBf16) return bf16r(v);
  if (MODE == kModeInt8) return quant_i8(v, inv_sx_next);
  return v;
}

// INT8 calibration (etx_calibrate; sec. 7.4, R21): max |x| over the existing rows of a
// Linear's input tile.  Called by all threads of the CTA once the tile is complete; max is order-free, and non-negative
// floats order like their bit patterns, so one integer atomicMax per warp keeps the running maximum.
template <int NT>
__device__ __forceinline__ void tile_absmax(float* slot, const float* X, int ld, int K, int rows) {
  float mx = 0.0f;
  for (int i = threadIdx.x; i < rows * K; i += NT) mx = fmaxf(mx, fabsf(X[(i / K) * ld + i % K]));
#pragma unroll
  for (int o = 16; o; o >>= 1) mx = fmaxf(mx, __shfl_xor_sync(0xffffffffu, mx, o));
  if ((threadIdx.x & 31) == 0 && mx > 0.0f) atomicMax(reinterpret_cast<int*>(slot), __float_as_int(mx));
}

// ---- one dense layer over a tile of R rows held in shared memory -----------------------------------------
// 256 threads; thread (rg, cg) owns the TM rows rg, rg + RG, rg + 2 RG, ... x 4 consecutive output columns (rows
// interleaved, so the two row groups of a warp read neighbouring rows of X: different banks whatever TM is).
// X: [R][ldx] fp32 in shared memory (ldx % 4 == 0), Wt: [K][N] in shared memory (the GNN kernels stage both weight
// matrices once per CTA) or in global memory (L1-resident: embedding, triplet classifiers).
// epi(row_in_tile, col, acc[4]).  Blocking over rows and output channels only changes which thread owns an output:
// each output is still ONE ascending-k fmaf chain (R3), so the result does not depend on the tile shape.
template <int N, int R, int NT = kMlpThreads, typename Epi>
__device__ __forceinline__ void dense_tile(const float* __restrict__ X, int ldx, int K,
                                           const float* __restrict__ Wt, Epi epi) {
  constexpr int CG = N / 4, RG = NT / CG, TM = R / RG;
  static_assert(TM >= 1 && RG * TM == R, "tile shape");
  const int cg = threadIdx.x % CG, rg = threadIdx.x / CG;
  float acc[TM][4];
#pragma unroll
  for (int i = 0; i < TM; ++i) acc[i][0] = acc[i][1] = acc[i][2] = acc[i][3] = 0.0f;
  const float* xr = X + (size_t)rg * ldx;
  const int rstep = RG * ldx;
  const float4* w4 = reinterpret_cast<const float4*>(Wt) + cg;
  int k = 0;
  for (; k + 4 <= K; k += 4) {
    const float4 w0 = w4[(size_t)(k + 0) * CG], w1 = w4[(size_t)(k + 1) * CG],
                 w2 = w4[(size_t)(k + 2) * CG], w3 = w4[(size_t)(k + 3) * CG];
#pragma unroll
    for (int i = 0; i < TM; ++i) {
      const float4 x = *reinterpret_cast<const float4*>(xr + i * rstep + k);
      acc[i][0] = __fmaf_rn(x.x, w0.x, acc[i][0]); acc[i][1] = __fmaf_rn(x.x, w0.y, acc[i][1]);
      acc[i][2] = __fmaf_rn(x.x, w0.z, acc[i][2]); acc[i][3] = __fmaf_rn(x.x, w0.w, acc[i][3]);
      acc[i][0] = __fmaf_rn(x.y, w1.x, acc[i][0]); acc[i][1] = __fmaf_rn(x.y, w1.y, acc[i][1]);
      acc[i][2] = __fmaf_rn(x.y, w1.z, acc[i][2]); acc[i][3] = __fmaf_rn(x.y, w1.w, acc[i][3]);
      acc[i][0] = __fmaf_rn(x.z, w2.x, acc[i][0]); acc[i][1] = __fmaf_rn(x.z, w2.y, acc[i][1]);
      acc[i][2] = __fmaf_rn(x.z, w2.z, acc[i][2]); acc[i][3] = __fmaf_rn(x.z, w2.w, acc[i][3]);
      acc[i][0] = __fmaf_rn(x.w, w3.x, acc[i][0]); acc[i][1] = __fmaf_rn(x.w, w3.y, acc[i][1]);
      acc[i][2] = __fmaf_rn(x.w, w3.z, acc[i][2]); acc[i][3] = __fmaf_rn(x.w, w3.w, acc[i][3]);
    }
  }
  for (; k < K; ++k) {
    const float4 w0 = w4[(size_t)k * CG];
#pragma unroll
    for (int i = 0; i < TM; ++i) {
      const float x = xr[i * rstep + k];
      acc[i][0] = __fmaf_rn(x, w0.x, acc[i][0]); acc[i][1] = __fmaf_rn(x, w0.y, acc[i][1]);
      acc[i][2] = __fmaf_rn(x, w0.z, acc[i][2]); acc[i][3] = __fmaf_rn(x, w0.w, acc[i][3]);
    }
  }
#pragma unroll
  for (int i = 0; i < TM; ++i) epi(rg + i * RG, cg * 4, acc[i]);
}

// K = 3 input layer (never a tensor layer): out[r][c] = relu(fmaf chain + b), converted for the next layer.
template <int MODE, int R, int NT = kMlpThreads>
__device__ __forceinline__ void input_layer3(const float* __restrict__ F /*[R][4] smem*/, const LayerP& L,
                                             float inv_sx_next, float* __restrict__ Y, int ldy) {
  const int N = L.N;
  for (int idx = threadIdx.x; idx < R * N; idx += NT) {
    const int r = idx / N, c = idx % N;
    float acc = 0.0f;
    acc = __fmaf_rn(F[r * 4 + 0], __ldg(L.Wt + c), acc);
    acc = __fmaf_rn(F[r * 4 + 1], __ldg(L.Wt + N + c), acc);
    acc = __fmaf_rn(F[r * 4 + 2], __ldg(L.Wt + 2 * N + c), acc);
    float y = __fadd_rn(acc, __ldg(L.bias + c));
    y = y > 0.0f ? y : 0.0f;
    Y[r * ldy + c] = to_operand<MODE>(y, inv_sx_next);
  }
}

// ============================================================================================================
// S1: hit-embedding MLP (sec. 5.1; R2, R3): 3 -> D -> ... -> D -> 4, ReLU on hidden layers only.
template <int MODE, int D>
__global__ void __launch_bounds__(kMlpThreads) embed_simt_kernel(EmbArgs a) {
  constexpr int R = kTileRows, LD = D + 4;
  extern __shared__ __align__(16) float smem[];
  float* A = smem;                 // [R][LD]
  float* B = smem + R * LD;        // [R][LD]
  float* F = B + R * LD;           // [R][4]
  const int H = a.n_layers - 1;
  for (int tile = blockIdx.x; tile * R < a.n_rows; tile += gridDim.x) {
    const int row0 = tile * R;
    __syncthreads();
    if (threadIdx.x < R) {
      const int row = row0 + threadIdx.x;
      float4 f = row < a.n_rows ? a.feat[row] : make_float4(0.f, 0.f, 0.f, 0.f);
      *reinterpret_cast<float4*>(F + threadIdx.x * 4) = f;
    }
    __syncthreads();
    input_layer3<MODE, R>(F, a.layers[0], a.layers[1].inv_sx, A, LD);
    __syncthreads();
    const int rows_here = min(R, a.n_rows - row0);
    if (a.absmax) tile_absmax<kMlpThreads>(a.absmax + a.layers[1].index, A, LD, a.layers[1].K, rows_here);
    float* cur = A; float* nxt = B;
    for (int l = 1; l < H; ++l) {
      const LayerP L = a.layers[l];
      const float inv_next = a.layers[l + 1].inv_sx;
      int32_t* tap = (a.tap && a.tap_layer == L.index) ? a.tap : nullptr;
      dense_tile<D, R>(cur, LD, L.K, L.Wt, [&](int r, int c, const float* acc) {
        float4 sc = __ldg(reinterpret_cast<const float4*>(L.scale + c)), bi = __ldg(reinterpret_cast<const float4*>(L.bias + c));
        float y[4] = {__fmaf_rn(acc[0], sc.x, bi.x), __fmaf_rn(acc[1], sc.y, bi.y), __fmaf_rn(acc[2], sc.z, bi.z), __fmaf_rn(acc[3], sc.w, bi.w)};
#pragma unroll
        for (int j = 0; j < 4; ++j) { y[j] = y[j] > 0.0f ? y[j] : 0.0f; y[j] = to_operand<MODE>(y[j], inv_next); }
        *reinterpret_cast<float4*>(nxt + r * LD + c) = make_float4(y[0], y[1], y[2], y[3]);
        if (tap && row0 + r < a.n_rows)
          for (int j = 0; j < 4; ++j) tap[(size_t)(row0 + r) * D + c + j] = (int32_t)acc[j];
      });
      __syncthreads();
      float* t = cur; cur = nxt; nxt = t;
      if (a.absmax) tile_absmax<kMlpThreads>(a.absmax + a.layers[l + 1].index, cur, LD, a.layers[l + 1].K, rows_here);
    }
    // output layer D -> 4, linear, fp32 result (R20: the embedding output is not rounded)
    {
      const LayerP L = a.layers[H];
      const int r = threadIdx.x / 4, c = threadIdx.x % 4;       // R * 4 == 256 threads
      float acc = 0.0f;
      const float* x = cur + r * LD;
      for (int j = 0; j < L.K; ++j) acc = __fmaf_rn(x[j], __ldg(L.Wt + j * 4 + c), acc);
      const float y = __fmaf_rn(acc, __ldg(L.scale + c), __ldg(L.bias + c));
      if (row0 + r < a.n_rows) {
        reinterpret_cast<float*>(a.emb)[(size_t)(row0 + r) * 4 + c] = y;
        if (a.tap && a.tap_layer == L.index) a.tap[(size_t)(row0 + r) * 4 + c] = (int32_t)acc;
      }
    }
  }
}

// ============================================================================================================
// S4a/b/d/e (+ S4f): the four two-layer MLPs of the interaction network (sec. 5.2).
//   node encoder  h0 = MLP(f)                                   (L133)
//   edge encoder  e0 = MLP(|f_dst - f_src|)  or MLP([h0_s,h0_d]) (R10, R11)
//   node network  h <- h + MLP([h, m_out, m_in])                (L140, R12, R14)
//   edge network  e <- e + MLP([h_src, h_dst, e]), updated h    (L140, R13); optional head z = w.e + b (R16)
template <int KIND, int MODE, typename ST, int D>
__global__ void __launch_bounds__(kGnnThreads) gnn_mlp_simt_kernel(GnnArgs a) {
  // 128-row tiles, 8 rows x 4 output channels per thread, both weight matrices resident in shared memory (128 FFMA per
  // 12 conflict-free shared-memory loads), and the gather of the input rows issued eight loads deep per thread.  The
  // 64-row kernel with weights read through L1 ran at 30 % of the FFMA pipe; what held it back was the gather, one
  // dependent load per loop iteration (profiles/r2_kernels_full.md).
  constexpr int R = kGnnRows;
  constexpr int K0MAX = 3 * D, LDX = K0MAX + 4, LDY = D + 4;
  extern __shared__ __align__(16) float smem[];
  float* X = smem;                       // [R][LDX]
  float* Y = X + R * LDX;                // [R][LDY]
  float* W0s = Y + R * LDY;              // [K0][D]   layer-0 weights (tensor layers; a K = 3 layer reads its own through L1)
  float* W1s = W0s + K0MAX * D;          // [D][D]
  int* IDX = reinterpret_cast<int*>(W1s + D * D);   // [2][R] src, dst
  const int n_rows = a.n_rows_ptr ? *a.n_rows_ptr : a.n_rows;
  const bool is_edge = (KIND == kEdgeEnc || KIND == kEdgeNet);
  const LayerP L0 = a.l0, L1 = a.l1;
  const bool quant_in = (MODE == kModeInt8) && L0.tensor;
  if (L0.K > 3) for (int i = threadIdx.x; i < L0.K * D / 4; i += kGnnThreads) reinterpret_cast<float4*>(W0s)[i] = __ldg(reinterpret_cast<const float4*>(L0.Wt) + i);
  for (int i = threadIdx.x; i < D * D / 4; i += kGnnThreads) reinterpret_cast<float4*>(W1s)[i] = __ldg(reinterpret_cast<const float4*>(L1.Wt) + i);

  for (int tile = blockIdx.x; (size_t)tile * R < (size_t)n_rows; tile += gridDim.x) {
    const int row0 = tile * R;
    __syncthreads();
    if (is_edge && threadIdx.x < 2 * R) {
      const int r = threadIdx.x % R, which = threadIdx.x / R;
      const int row = row0 + r;
      IDX[which * R + r] = row < n_rows ? (which ? a.dst[row] : a.src[row]) : 0;
    }
    __syncthreads();
    // ---- assemble the layer-0 input ------------------------------------------------------------------------
    if (KIND == kNodeEnc || (KIND == kEdgeEnc && a.edge_enc_input == 0)) {
      if (threadIdx.x < R) {
        const int r = threadIdx.x, row = row0 + r;
        float4 f = make_float4(0.f, 0.f, 0.f, 0.f);
        if (row < n_rows) {
          if (KIND == kNodeEnc) f = a.feat[row];
          else {
            const float4 fs = a.feat[IDX[r]], fd = a.feat[IDX[R + r]];
            f = make_float4(fabsf(__fsub_rn(fd.x, fs.x)), fabsf(__fsub_rn(fd.y, fs.y)), fabsf(__fsub_rn(fd.z, fs.z)), 0.f);
          }
        }
        *reinterpret_cast<float4*>(Y + r * 4) = f;       // Y doubles as the [R][4] feature buffer
      }
      __syncthreads();
      // layer 0 (K = 3) writes its output (the layer-1 operand) into X, then Y is free again
      input_layer3<MODE, R, kGnnThreads>(Y, L0, L1.inv_sx, X, LDX);
      __syncthreads();
      if (a.absmax) tile_absmax<kGnnThreads>(a.absmax + L1.index, X, LDX, D, min(R, n_rows - row0));
    } else {
      const int K0 = L0.K;                               // 2D (paper's edge encoder) or 3D
      const int c4n = K0 / 4, seg4 = D / 4;
      constexpr int GB = 8;                              // loads in flight per thread
      for (int base = 0; base < R * c4n; base += kGnnThreads * GB) {
        float4 v[GB];
#pragma unroll
        for (int u = 0; u < GB; ++u) {
          const int idx = base + u * kGnnThreads + threadIdx.x;
          v[u] = make_float4(0.f, 0.f, 0.f, 0.f);
          if (idx < R * c4n) {
            const int r = idx / c4n, c4 = idx % c4n, seg = c4 / seg4, within = (c4 % seg4) * 4;
            const int row = row0 + r;
            if (row < n_rows) {
              if (KIND == kNodeNet) {
                v[u] = seg == 0 ? State<ST>::ld4(a.h, (size_t)row * D + within)
                                : State<ST>::ld4(a.m, (size_t)row * 2 * D + (size_t)(seg - 1) * D + within);
              } else {
                if (seg == 0) v[u] = State<ST>::ld4(a.h, (size_t)IDX[r] * D + within);
                else if (seg == 1) v[u] = State<ST>::ld4(a.h, (size_t)IDX[R + r] * D + within);
                else v[u] = State<ST>::ld4(a.e, (size_t)row * D + within);
              }
            }
          }
        }
#pragma unroll
        for (int u = 0; u < GB; ++u) {
          const int idx = base + u * kGnnThreads + threadIdx.x;
          if (idx < R * c4n) {
            float4 w = v[u];
            if (quant_in) { w.x = quant_i8(w.x, L0.inv_sx); w.y = quant_i8(w.y, L0.inv_sx); w.z = quant_i8(w.z, L0.inv_sx); w.w = quant_i8(w.w, L0.inv_sx); }
            *reinterpret_cast<float4*>(X + (idx / c4n) * LDX + (idx % c4n) * 4) = w;
          }
        }
      }
      __syncthreads();
      if (a.absmax) tile_absmax<kGnnThreads>(a.absmax + L0.index, X, LDX, K0, min(R, n_rows - row0));
      // layer 0: K0 -> D, ReLU, operand conversion for layer 1
      int32_t* tap0 = (a.tap && a.tap_layer == L0.index) ? a.tap : nullptr;
      dense_tile<D, R, kGnnThreads>(X, LDX, K0, W0s, [&](int r, int c, const float* acc) {
        float4 sc = __ldg(reinterpret_cast<const float4*>(L0.scale + c)), bi = __ldg(reinterpret_cast<const float4*>(L0.bias + c));
        float y[4] = {__fmaf_rn(acc[0], sc.x, bi.x), __fmaf_rn(acc[1], sc.y, bi.y), __fmaf_rn(acc[2], sc.z, bi.z), __fmaf_rn(acc[3], sc.w, bi.w)};
#pragma unroll
        for (int j = 0; j < 4; ++j) { y[j] = y[j] > 0.0f ? y[j] : 0.0f; y[j] = to_operand<MODE>(y[j], L1.inv_sx); }
        *reinterpret_cast<float4*>(Y + r * LDY + c) = make_float4(y[0], y[1], y[2], y[3]);
        if (tap0 && row0 + r < n_rows)
          for (int j = 0; j < 4; ++j) tap0[(size_t)(row0 + r) * D + c + j] = (int32_t)acc[j];
      });
      __syncthreads();
      if (a.absmax) tile_absmax<kGnnThreads>(a.absmax + L1.index, Y, LDY, D, min(R, n_rows - row0));
    }
    const bool hidden_in_x = (KIND == kNodeEnc || (KIND == kEdgeEnc && a.edge_enc_input == 0));
    const float* HID = hidden_in_x ? X : Y;
    const int ldh = hidden_in_x ? LDX : LDY;
    float* OUT = hidden_in_x ? Y : X;           // staging of the new state rows for the fused head
    const int ldo = hidden_in_x ? LDY : LDX;
    // ---- layer 1: D -> D, linear; residual for the networks; store the state --------------------------------
    int32_t* tap1 = (a.tap && a.tap_layer == L1.index) ? a.tap : nullptr;
    void* state = is_edge ? a.e : a.h;
    dense_tile<D, R, kGnnThreads>(HID, ldh, D, W1s, [&](int r, int c, const float* acc) {
      const int row = row0 + r;
      float4 sc = __ldg(reinterpret_cast<const float4*>(L1.scale + c)), bi = __ldg(reinterpret_cast<const float4*>(L1.bias + c));
      float4 y = make_float4(__fmaf_rn(acc[0], sc.x, bi.x), __fmaf_rn(acc[1], sc.y, bi.y), __fmaf_rn(acc[2], sc.z, bi.z), __fmaf_rn(acc[3], sc.w, bi.w));
      if (row < n_rows) {
        if (KIND == kNodeNet || KIND == kEdgeNet) {
          const float4 old = State<ST>::ld4(state, (size_t)row * D + c);
          y = make_float4(__fadd_rn(old.x, y.x), __fadd_rn(old.y, y.y), __fadd_rn(old.z, y.z), __fadd_rn(old.w, y.w));
        }
        y = make_float4(State<ST>::round(y.x), State<ST>::round(y.y), State<ST>::round(y.z), State<ST>::round(y.w));
        State<ST>::st4(state, (size_t)row * D + c, y);
        if (tap1) for (int j = 0; j < 4; ++j) tap1[(size_t)row * D + c + j] = (int32_t)acc[j];
      }
      if (is_edge && a.do_head) *reinterpret_cast<float4*>(OUT + r * ldo + c) = y;
    });
    // ---- S4f: edge classifier on the final edge state (L80, L142; R16): z = w.e + b, score = sigmoid(z) -----
    if (is_edge && a.do_head) {
      __syncthreads();
      if (threadIdx.x < R && row0 + threadIdx.x < n_rows) {
        const float* x = OUT + threadIdx.x * ldo;
        float acc = 0.0f;
        for (int j = 0; j < D; ++j) acc = __fmaf_rn(x[j], __ldg(a.head.Wt + j), acc);
        const float z = __fadd_rn(acc, __ldg(a.head.bias));
        a.logit[row0 + threadIdx.x] = z;
        a.score[row0 + threadIdx.x] = 1.0f / (1.0f + expf(-z));
      }
    }
  }
}

// ============================================================================================================
// S4c: message building, Eq.(4): m_l = [ sum_{l->j} e_lj , sum_{i->l} e_il ].
// The paper needed a scatter_add TensorRT plugin (global atomics, L253).  Here nothing is scattered: the
// out-edges of a node are a contiguous run of e (edges are src-sorted) and its in-edges are listed by the
// CSC, so each node's sums are sequential fp32 adds in ascending edge id (R22) -- deterministic, no atomics.
// One group of lanes per node, 16 bytes of the row per lane (8 bf16 or 4 fp32 columns).  The pass is bound by
// instruction issue as much as by bytes (ncu: 61 % of the issue slots at 69 % of the HBM peak with 8-byte loads), so
// the widest load is what counts.
template <typename ST> struct Vec16;
template <> struct Vec16<float> {
  static constexpr int V = 4;
  static __device__ __forceinline__ void add(const void* base, size_t elem, float (&s)[4]) {
    const float4 v = *reinterpret_cast<const float4*>(static_cast<const float*>(base) + elem);
    s[0] = __fadd_rn(s[0], v.x); s[1] = __fadd_rn(s[1], v.y); s[2] = __fadd_rn(s[2], v.z); s[3] = __fadd_rn(s[3], v.w);
  }
  static __device__ __forceinline__ void st(void* base, size_t elem, const float (&x)[4]) {
    *reinterpret_cast<float4*>(static_cast<float*>(base) + elem) = make_float4(x[0], x[1], x[2], x[3]);
  }
};
template <> struct Vec16<__nv_bfloat16> {
  static constexpr int V = 8;
  static __device__ __forceinline__ void add(const void* base, size_t elem, float (&s)[8]) {
    const uint4 u = *reinterpret_cast<const uint4*>(static_cast<const __nv_bfloat16*>(base) + elem);
    s[0] = __fadd_rn(s[0], __uint_as_float(u.x << 16)); s[1] = __fadd_rn(s[1], __uint_as_float(u.x & 0xffff0000u));
    s[2] = __fadd_rn(s[2], __uint_as_float(u.y << 16)); s[3] = __fadd_rn(s[3], __uint_as_float(u.y & 0xffff0000u));
    s[4] = __fadd_rn(s[4], __uint_as_float(u.z << 16)); s[5] = __fadd_rn(s[5], __uint_as_float(u.z & 0xffff0000u));
    s[6] = __fadd_rn(s[6], __uint_as_float(u.w << 16)); s[7] = __fadd_rn(s[7], __uint_as_float(u.w & 0xffff0000u));
  }
  static __device__ __forceinline__ void st(void* base, size_t elem, const float (&x)[8]) {   // RNE to bf16 (R20)
    uint4 u;
    u.x = (__float_as_uint(bf16r(x[0])) >> 16) | (__float_as_uint(bf16r(x[1])) & 0xffff0000u);
    u.y = (__float_as_uint(bf16r(x[2])) >> 16) | (__float_as_uint(bf16r(x[3])) & 0xffff0000u);
    u.z = (__float_as_uint(bf16r(x[4])) >> 16) | (__float_as_uint(bf16r(x[5])) & 0xffff0000u);
    u.w = (__float_as_uint(bf16r(x[6])) >> 16) | (__float_as_uint(bf16r(x[7])) & 0xffff0000u);
    *reinterpret_cast<uint4*>(static_cast<__nv_bfloat16*>(base) + elem) = u;
  }
};

// 64-thread blocks: 1.81 ms for the six launches at cfg 2 against 1.83-1.88 (128) and 1.85-1.93 (256), same box -- the
// shorter the block, the smaller the tail behind its longest node
constexpr int kScatterThreads = 64;

template <typename ST, int D>
__global__ void __launch_bounds__(kScatterThreads) scatter_kernel(const void* __restrict__ e, const int32_t* __restrict__ row_ptr,
                                                      const int32_t* __restrict__ col_ptr, const int32_t* __restrict__ in_edge,
                                                      void* __restrict__ m, int n_hits) {
  constexpr int V = Vec16<ST>::V, LPN = D / V;            // lanes per node
  // Nodes are walked from the last to the first: the edge network that ran just before wrote e in ascending
  // order, so the tail of e is what the L2 still holds, and the next edge network starts at the head, which this
  // pass reads last.
  const int gid = (gridDim.x - 1 - blockIdx.x) * (kScatterThreads / LPN) + threadIdx.x / LPN;
  const int c = (threadIdx.x % LPN) * V;
  if (gid >= n_hits) return;
  float sum[V];
#pragma unroll
  for (int j = 0; j < V; ++j) sum[j] = 0.0f;
  const int a0 = row_ptr[gid], a1 = row_ptr[gid + 1];
  const int b0 = col_ptr[gid], b1 = col_ptr[gid + 1];
  for (int i = a0; i < a1; ++i) Vec16<ST>::add(e, (size_t)i * D + c, sum);
  Vec16<ST>::st(m, (size_t)gid * 2 * D + c, sum);         // m_out is stored before m_in starts: one live accumulator set
#pragma unroll
  for (int j = 0; j < V; ++j) sum[j] = 0.0f;
  for (int i = b0; i < b1; ++i) Vec16<ST>::add(e, (size_t)in_edge[i] * D + c, sum);
  Vec16<ST>::st(m, (size_t)gid * 2 * D + D + c, sum);
}

// ------------------------------------------------------------------------------------------------------------
template <int D> static size_t gnn_smem() {
  return sizeof(float) * (kGnnRows * ((3 * D + 4) + (D + 4)) + 3 * D * D + D * D) + sizeof(int) * 2 * kGnnRows;
}
template <int D> static size_t emb_smem() { return sizeof(float) * kTileRows * (2 * (D + 4) + 4); }

template <int KIND, int MODE, typename ST, int D>
static void gnn_launch_one(etx_ctx* c, const GnnArgs& a, int max_rows, cudaStream_t s) {
  auto kern = gnn_mlp_simt_kernel<KIND, MODE, ST, D>;
  opt_in_smem(c, kern, (int)gnn_smem<D>());
  const int tiles = (max_rows + kGnnRows - 1) / kGnnRows;
  int per_sm = (int)((227 * 1024) / (gnn_smem<D>() + 1024));
  if (per_sm < 1) per_sm = 1;
  const int grid = tiles < c->sm_count * per_sm ? tiles : c->sm_count * per_sm;
  if (grid <= 0) return;
  kern<<<grid, kGnnThreads, gnn_smem<D>(), s>>>(a);
  c->launches++;
}

template <int MODE, typename ST, int D>
static void gnn_launch_kind(etx_ctx* c, int kind, const GnnArgs& a, int max_rows, cudaStream_t s) {
  switch (kind) {
    case kNodeEnc: gnn_launch_one<kNodeEnc, MODE, ST, D>(c, a, max_rows, s); break;
    case kEdgeEnc: gnn_launch_one<kEdgeEnc, MODE, ST, D>(c, a, max_rows, s); break;
    case kNodeNet: gnn_launch_one<kNodeNet, MODE, ST, D>(c, a, max_rows, s); break;
    default:       gnn_launch_one<kEdgeNet, MODE, ST, D>(c, a, max_rows, s); break;
  }
}

template <int D>
static void gnn_launch_d(etx_ctx* c, int kind, const GnnArgs& a, int max_rows, cudaStream_t s) {
  if (c->precision == ETX_FP32) gnn_launch_kind<kModeF32, float, D>(c, kind, a, max_rows, s);
  else if (c->precision == ETX_BF16) gnn_launch_kind<kModeBf16, __nv_bfloat16, D>(c, kind, a, max_rows, s);
  else if (c->state_bf16) gnn_launch_kind<kModeInt8, __nv_bfloat16, D>(c, kind, a, max_rows, s);   // R21 with state_dtype = bf16
  else gnn_launch_kind<kModeInt8, float, D>(c, kind, a, max_rows, s);
}

void fill_gnn_args(etx_ctx* c, int kind, int iter, int n_hits, bool do_head, GnnArgs& a) {
  const bool is_edge = (kind == kEdgeEnc || kind == kEdgeNet);
  int i0;
  if (kind == kNodeEnc) i0 = c->i_nenc;
  else if (kind == kEdgeEnc) i0 = c->i_eenc;
  else if (kind == kNodeNet) i0 = c->i_iter0 + 4 * iter;
  else i0 = c->i_iter0 + 4 * iter + 2;
  a.l0 = c->layers[i0].dev; a.l1 = c->layers[i0 + 1].dev; a.head = c->layers[c->i_head].dev;
  a.feat = c->feat; a.src = c->src; a.dst = c->dst;
  a.n_rows_ptr = is_edge ? c->n_edges : nullptr;
  a.n_rows = n_hits;
  a.h = c->h; a.e = c->e; a.m = c->m; a.logit = c->logit; a.score = c->score_out;
  a.do_head = do_head ? 1 : 0;
  a.edge_enc_input = c->hp.edge_enc_input;
  a.tap = c->tap_layer >= 0 ? c->tap : nullptr;
  a.tap_layer = c->tap_layer;
  a.absmax = c->calibrating ? c->absmax : nullptr;
}

void launch_gnn_mlp_simt(etx_ctx* c, int kind, int iter, int n_hits, bool do_head, cudaStream_t s) {
  GnnArgs a;
  fill_gnn_args(c, kind, iter, n_hits, do_head, a);
  const bool is_edge = (kind == kEdgeEnc || kind == kEdgeNet);
  // edge kernels: E is only known on the device; size the grid for the capacity k * n_hits
  const long long max_rows_ll = is_edge ? (long long)n_hits * c->hp.k : n_hits;
  const int max_rows = (int)(max_rows_ll > 0x7fffffff ? 0x7fffffff : max_rows_ll);
  if (c->hp.gnn_latent == 32) gnn_launch_d<32>(c, kind, a, max_rows, s);
  else gnn_launch_d<64>(c, kind, a, max_rows, s);
}

template <int MODE, int D>
static void emb_launch(etx_ctx* c, const EmbArgs& a, cudaStream_t s) {
  auto kern = embed_simt_kernel<MODE, D>;
  opt_in_smem(c, kern, (int)emb_smem<D>());
  const int tiles = (a.n_rows + kTileRows - 1) / kTileRows;
  const int grid = tiles < c->sm_count * 3 ? tiles : c->sm_count * 3;
  if (grid <= 0) return;
  kern<<<grid, kMlpThreads, emb_smem<D>(), s>>>(a);
  c->launches++;
}

void launch_embed_simt(etx_ctx* c, int n_hits, cudaStream_t s) {
  EmbArgs a;
  a.n_layers = c->hp.emb_n_hidden_layers + 1;
  for (int l = 0; l < a.n_layers; ++l) a.layers[l] = c->layers[c->i_emb0 + l].dev;
  a.feat = c->feat_emb; a.emb = c->emb; a.n_rows = n_hits;
  a.tap = c->tap_layer >= 0 ? c->tap : nullptr; a.tap_layer = c->tap_layer;
  a.absmax = c->calibrating ? c->absmax : nullptr;
  const int D = c->hp.emb_hidden;
#define ETX_EMB(MODE)                                   \
  if (D == 64) emb_launch<MODE, 64>(c, a, s);           \
  else emb_launch<MODE, 128>(c, a, s);
  if (c->precision == ETX_FP32) { ETX_EMB(kModeF32) }
  else if (c->precision == ETX_BF16) { ETX_EMB(kModeBf16) }
  else { ETX_EMB(kModeInt8) }
#undef ETX_EMB
}

void launch_scatter(etx_ctx* c, int n_hits, cudaStream_t s) {
  if (n_hits == 0) return;
  const int d = c->hp.gnn_latent;
  const int npb = kScatterThreads / (d / (c->state_bf16 ? 8 : 4));
  const int grid = (n_hits + npb - 1) / npb;
  if (c->state_bf16) {
    if (d == 32) scatter_kernel<__nv_bfloat16, 32><<<grid, kScatterThreads, 0, s>>>(c->e, c->row_ptr, c->col_ptr, c->in_edge, c->m, n_hits);
    else scatter_kernel<__nv_bfloat16, 64><<<grid, kScatterThreads, 0, s>>>(c->e, c->row_ptr, c->col_ptr, c->in_edge, c->m, n_hits);
  } else {
    if (d == 32) scatter_kernel<float, 32><<<grid, kScatterThreads, 0, s>>>(c->e, c->row_ptr, c->col_ptr, c->in_edge, c->m, n_hits);
    else scatter_kernel<float, 64><<<grid, kScatterThreads, 0, s>>>(c->e, c->row_ptr, c->col_ptr, c->in_edge, c->m, n_hits);
  }
  c->launches++;
}

// ============================================================================================================
// Triplet classifier (R28): z = w1 . relu(W0 [e_first, e_second] + b0) + b1 on pairs of
// FINAL edge encodings, one classifier for articulations and one for elbows.  The 2d -> d layer is a tensor layer in
// the sense of R20 / R21 (bf16 weights and rounded hidden activation / int8 codes), the d -> 1 layer is fp32 in the
// pinned order like the edge head.  Same arithmetic in every precision as the rest of this file, so fp32 and int8
// are bit-exact against the oracle.
struct TripArgs {
  LayerP l0, l1;
  const void* e;                // [E][d] final edge state, state dtype
  const int32_t* first; const int32_t* second;
  const int32_t* n_ptr;         // device count of this kind
  int cap;
  float* logit; float* score;
  float* absmax;                // calibration: running max |x| per layer (blob order), or nullptr
};

template <int MODE, typename ST, int D>
__global__ void __launch_bounds__(kMlpThreads) triplet_cls_simt_kernel(TripArgs a) {
  constexpr int R = kTileRows, LDX = 2 * D + 4, LDY = D + 4;
  extern __shared__ __align__(16) float smem[];
  float* X = smem;                       // [R][LDX]
  float* Y = X + R * LDX;                // [R][LDY]
  const int n_rows = min(*a.n_ptr, a.cap);
  const LayerP L0 = a.l0, L1 = a.l1;
  for (int tile = blockIdx.x; (size_t)tile * R < (size_t)n_rows; tile += gridDim.x) {
    const int row0 = tile * R;
    __syncthreads();
    constexpr int c4n = 2 * D / 4, seg4 = D / 4;
    for (int idx = threadIdx.x; idx < R * c4n; idx += kMlpThreads) {
      const int r = idx / c4n, c4 = idx % c4n, seg = c4 / seg4, within = (c4 % seg4) * 4;
      const int row = row0 + r;
      float4 v = make_float4(0.f, 0.f, 0.f, 0.f);
      if (row < n_rows) v = State<ST>::ld4(a.e, (size_t)(seg ? a.second[row] : a.first[row]) * D + within);
      if (MODE == kModeInt8) { v.x = quant_i8(v.x, L0.inv_sx); v.y = quant_i8(v.y, L0.inv_sx); v.z = quant_i8(v.z, L0.inv_sx); v.w = quant_i8(v.w, L0.inv_sx); }
      *reinterpret_cast<float4*>(X + r * LDX + c4 * 4) = v;
    }
    __syncthreads();
    if (a.absmax) tile_absmax<kMlpThreads>(a.absmax + L0.index, X, LDX, 2 * D, min(R, n_rows - row0));
    dense_tile<D, R>(X, LDX, 2 * D, L0.Wt, [&](int r, int c, const float* acc) {
      float4 sc = __ldg(reinterpret_cast<const float4*>(L0.scale + c)), bi = __ldg(reinterpret_cast<const float4*>(L0.bias + c));
      float y[4] = {__fmaf_rn(acc[0], sc.x, bi.x), __fmaf_rn(acc[1], sc.y, bi.y), __fmaf_rn(acc[2], sc.z, bi.z), __fmaf_rn(acc[3], sc.w, bi.w)};
#pragma unroll
      for (int j = 0; j < 4; ++j) { y[j] = y[j] > 0.0f ? y[j] : 0.0f; if (MODE == kModeBf16) y[j] = bf16r(y[j]); }   // the next layer is fp32: no int8 codes
      *reinterpret_cast<float4*>(Y + r * LDY + c) = make_float4(y[0], y[1], y[2], y[3]);
    });
    __syncthreads();
    if (threadIdx.x < R && row0 + threadIdx.x < n_rows) {
      const float* x = Y + threadIdx.x * LDY;
      float acc = 0.0f;
      for (int j = 0; j < D; ++j) acc = __fmaf_rn(x[j], __ldg(L1.Wt + j), acc);
      const float z = __fadd_rn(acc, __ldg(L1.bias));
      a.logit[row0 + threadIdx.x] = z;
      a.score[row0 + threadIdx.x] = 1.0f / (1.0f + expf(-z));
    }
  }
}

template <int MODE, typename ST, int D>
static void trip_launch(etx_ctx* c, const TripArgs& a, cudaStream_t s) {
  auto kern = triplet_cls_simt_kernel<MODE, ST, D>;
  const int smem = (int)(sizeof(float) * kTileRows * (2 * D + 4 + D + 4));
  opt_in_smem(c, kern, smem);
  const int tiles = (a.cap + kTileRows - 1) / kTileRows;
  const int grid = tiles < c->sm_count * 3 ? tiles : c->sm_count * 3;
  if (grid <= 0) return;
  kern<<<grid, kMlpThreads, smem, s>>>(a);
  c->launches++;
}

// kind 0: articulations (classifier i_trip, i_trip + 1); kinds 1, 2: elbows (i_trip + 2, i_trip + 3)
void launch_triplet_classifier(etx_ctx* c, int kind, cudaStream_t s) {
  if (c->edge_tma) { launch_triplet_cls_tma(c, kind, s); return; }     // bf16, AUTO engine: the tcgen05 tile code
  TripArgs a;
  const int i0 = c->i_trip + (kind ? 2 : 0);
  a.l0 = c->layers[i0].dev; a.l1 = c->layers[i0 + 1].dev;
  a.e = c->e;
  const size_t cap = (size_t)c->hp.max_triplets;
  a.first = c->trip_first + kind * cap; a.second = c->trip_second + kind * cap;
  a.n_ptr = c->trip_total + kind; a.cap = c->hp.max_triplets;
  a.logit = c->trip_logit + kind * cap; a.score = c->trip_score + kind * cap;
  a.absmax = c->calibrating ? c->absmax : nullptr;
#define ETX_TRIP(MODE, ST) { if (c->hp.gnn_latent == 32) trip_launch<MODE, ST, 32>(c, a, s); else trip_launch<MODE, ST, 64>(c, a, s); }
  if (c->precision == ETX_FP32) ETX_TRIP(kModeF32, float)
  else if (c->precision == ETX_BF16) ETX_TRIP(kModeBf16, __nv_bfloat16)
  else if (c->state_bf16) ETX_TRIP(kModeInt8, __nv_bfloat16)
  else ETX_TRIP(kModeInt8, float)
#undef ETX_TRIP
}

void simt_configure(etx_ctx*) {}

}  // namespace etx
