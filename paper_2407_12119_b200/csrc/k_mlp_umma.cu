// tcgen05 / TMEM tensor-core kernels for the MLP stages S1 and S4 (bf16 and int8 precision modes).
//
// Every Linear with K >= 16 (R20/R21) is a 128-row x N tile GEMM on the 5th-generation tensor
// cores: A (activations, K-major) and B (weights W[N][K], K-major -- the blob's own orientation) live in
// shared memory in the canonical swizzled UMMA layout, the fp32 / int32 accumulator lives in TMEM, one
// elected thread issues tcgen05.mma, completion arrives on an mbarrier via tcgen05.commit, and the
// epilogue reads the accumulator with tcgen05.ld (lane = row, so one thread owns one row).
// The two layers of each network are chained without leaving the SM: epilogue 0 (bias, ReLU, conversion to
// the next operand format) writes the A tile of layer 1 straight into shared memory.  The gather of
// h[src], h[dst], e (and of [h, m_out, m_in]) is fused into the A-tile build; the residual add, the
// state store and the d->1 edge classifier are fused into the last epilogue.  Weights are copied once per
// CTA with cp.async.bulk (TMA bulk copy) and stay resident for the CTA's lifetime (persistent tile loop).
//
// Shared-memory operand layout (K-major, swizzle width KB = 32 / 64 / 128 bytes): a tile is a sequence of
// K-blocks, each [rows][KB bytes]; inside a K-block the 16-byte chunk index is XORed with address bits
// [7, 7+log2(KB/16)) (the Swizzle<B,4,3> pattern the UMMA descriptor's layout_type names); 8-row groups
// are KB*8 bytes apart (SBO).  One K-block holds exactly one gathered segment (h_src | h_dst | e), so the
// concatenation [h_src, h_dst, e] costs nothing.
#include <string.h>

#include "umma_common.cuh"

namespace etx {

namespace {

using namespace umma;


// ============================================================================================================
// S4: the four two-layer MLPs of the interaction network, one 128-row tile at a time.
struct UmmaGnnSmem {           // byte offsets inside the 1024-aligned dynamic shared memory
  int a, h, w0, w1, par, idx, bar, total;
};
template <int PREC, int D>
__host__ __device__ constexpr UmmaGnnSmem gnn_smem_layout() {
  constexpr int ESZ = PREC == kBf16 ? 2 : 1;
  constexpr int SEGB = D * ESZ;                              // one gathered segment = one K-block
  UmmaGnnSmem s{};
  s.a = 0;                                 // A tile of layer 0: 3 K-blocks [128][SEGB]
  s.h = s.a + 3 * kRows * SEGB;            // A tile of layer 1: 1 K-block
  s.w0 = s.h + kRows * SEGB;               // W0: 3 K-blocks [D][SEGB]
  s.w1 = s.w0 + 3 * D * SEGB;              // W1
  s.par = s.w1 + D * SEGB;                 // fp32 params: scale0, bias0, scale1, bias1, head w (5 x D), W0 of a K=3 layer (3 x D)
  s.idx = s.par + 8 * D * 4;               // src / dst indices of the tile
  s.bar = s.idx + 2 * kRows * 4;           // 2 mbarriers + tmem address
  s.total = s.bar + 32;
  return s;
}

// SB: the state rows h / e / m are bf16 (always in bf16 mode; in int8 mode when state_dtype = bf16, R21)
template <int KIND, int PREC, int D, bool SB>
__global__ void __launch_bounds__(kUmmaThreads) gnn_mlp_umma_kernel(GnnArgs a) {
  static_assert(PREC != kBf16 || SB, "bf16 precision stores bf16 state");
  constexpr int ESZ = PREC == kBf16 ? 2 : 1;
  constexpr int KB = D * ESZ;                                // swizzle width = segment bytes (32 / 64 / 128)
  constexpr int CPR = KB / 16;                               // 16-byte chunks per segment row
  constexpr UmmaGnnSmem L = gnn_smem_layout<PREC, D>();
  constexpr uint32_t TMEM_COLS = 2 * D < 32 ? 32 : 2 * D;    // acc0 | acc1
  extern __shared__ uint8_t smem_raw[];
  uint8_t* smem = reinterpret_cast<uint8_t*>((reinterpret_cast<uintptr_t>(smem_raw) + 1023) & ~(uintptr_t)1023);
  uint8_t* A = smem + L.a; uint8_t* H = smem + L.h;
  float* par = reinterpret_cast<float*>(smem + L.par);
  float *scale0 = par, *bias0 = par + D, *scale1 = par + 2 * D, *bias1 = par + 3 * D, *headw = par + 4 * D, *w3 = par + 5 * D;
  int* IDX = reinterpret_cast<int*>(smem + L.idx);
  uint64_t* bar_w = reinterpret_cast<uint64_t*>(smem + L.bar);
  uint64_t* bar_mma = bar_w + 1;
  uint32_t* tmem_slot = reinterpret_cast<uint32_t*>(bar_w + 2);

  const int tid = threadIdx.x, warp = tid >> 5;
  const bool is_edge = (KIND == kEdgeEnc || KIND == kEdgeNet);
  const bool l0_tensor = a.l0.tensor != 0;                   // false: K = 3 input layer on FFMA (encoders)
  const int nseg = l0_tensor ? a.l0.K / D : 0;               // 3 (networks) or 2 (paper's edge encoder)
  const int n_rows = a.n_rows_ptr ? *a.n_rows_ptr : a.n_rows;

  // ---- one-time setup: barriers, TMEM, resident weights -------------------------------------------------------
  if (tid == 0) {
    mbar_init(bar_w, 1); mbar_init(bar_mma, 1);
    fence_barrier_init();
  }
  if (warp == 0) tmem_alloc(tmem_slot, TMEM_COLS);
  for (int i = tid; i < D; i += kUmmaThreads) {
    scale0[i] = a.l0.scale[i]; bias0[i] = a.l0.bias[i]; scale1[i] = a.l1.scale[i]; bias1[i] = a.l1.bias[i];
    headw[i] = a.head.Wt[i];
    if (!l0_tensor) { w3[i] = a.l0.Wt[i]; w3[D + i] = a.l0.Wt[D + i]; w3[2 * D + i] = a.l0.Wt[2 * D + i]; }
  }
  tc_fence_before();
  __syncthreads();
  tc_fence_after();
  const uint32_t tmem = *tmem_slot;
  if (tid == 0) {
    const uint32_t b0 = l0_tensor ? (uint32_t)(nseg * D * KB) : 0u, b1 = (uint32_t)(D * KB);
    mbar_expect_tx(bar_w, b0 + b1);
    if (l0_tensor) bulk_g2s(smem + L.w0, a.l0.Wtc, b0, bar_w);
    bulk_g2s(smem + L.w1, a.l1.Wtc, b1, bar_w);
  }
  mbar_wait(bar_w, 0);
  const uint32_t idesc = make_idesc<PREC>(D);
  const uint32_t a_addr = smem_u32(A), h_addr = smem_u32(H), w0_addr = smem_u32(smem + L.w0), w1_addr = smem_u32(smem + L.w1);
  const uint32_t lane_base = (uint32_t)(warp * 32) << 16;
  uint32_t phase = 0;
  const float head_b = a.head.bias[0];
  const float inv_sx0 = a.l0.inv_sx, inv_sx1 = a.l1.inv_sx;

  for (int tile = blockIdx.x; (size_t)tile * kRows < (size_t)n_rows; tile += gridDim.x) {
    const int row0 = tile * kRows;
    const int row = row0 + tid;
    const bool live = row < n_rows;
    if (is_edge) {
      IDX[tid] = live ? a.src[row] : 0;
      IDX[kRows + tid] = live ? a.dst[row] : 0;
    }
    __syncthreads();     // IDX visible; also: every thread is past the previous tile's last shared-memory reads

    if (l0_tensor) {
      // ---- fused gather: segment s of row r -> K-block s of the A tile -------------------------------------------
      for (int s = 0; s < nseg; ++s) {
        uint8_t* blk = A + s * (kRows * KB);
        if (PREC == kBf16) {
          const __nv_bfloat16* base; int stride_el;          // state rows are bf16
#pragma unroll
          for (int i = 0; i < CPR; ++i) {
            const int c = i * kUmmaThreads + tid, r = c / CPR, piece = c % CPR;
            size_t srow;
            if (KIND == kNodeNet) { base = static_cast<const __nv_bfloat16*>(s == 0 ? a.h : a.m); stride_el = s == 0 ? D : 2 * D; srow = (size_t)(row0 + r); }
            else if (s == 2) { base = static_cast<const __nv_bfloat16*>(a.e); stride_el = D; srow = (size_t)(row0 + r); }
            else { base = static_cast<const __nv_bfloat16*>(a.h); stride_el = D; srow = (size_t)IDX[s * kRows + r]; }
            const int col0 = (KIND == kNodeNet && s == 2) ? D : 0;
            uint4 v = make_uint4(0u, 0u, 0u, 0u);
            if (row0 + r < n_rows) v = __ldg(reinterpret_cast<const uint4*>(base + srow * stride_el + col0) + piece);
            *reinterpret_cast<uint4*>(blk + swz<KB>(r, piece)) = v;
          }
        } else if (SB) {
          const __nv_bfloat16* base; int stride_el;          // state rows are bf16: widen, quantise while gathering
#pragma unroll
          for (int i = 0; i < CPR; ++i) {
            const int c = i * kUmmaThreads + tid, r = c / CPR, piece = c % CPR;
            size_t srow;
            if (KIND == kNodeNet) { base = static_cast<const __nv_bfloat16*>(s == 0 ? a.h : a.m); stride_el = s == 0 ? D : 2 * D; srow = (size_t)(row0 + r); }
            else if (s == 2) { base = static_cast<const __nv_bfloat16*>(a.e); stride_el = D; srow = (size_t)(row0 + r); }
            else { base = static_cast<const __nv_bfloat16*>(a.h); stride_el = D; srow = (size_t)IDX[s * kRows + r]; }
            const int col0 = (KIND == kNodeNet && s == 2) ? D : 0;
            uint4 q = make_uint4(0u, 0u, 0u, 0u);
            if (row0 + r < n_rows) {
              const uint4* p = reinterpret_cast<const uint4*>(base + srow * stride_el + col0 + piece * 16);
              const uint4 u0 = __ldg(p), u1 = __ldg(p + 1);
              q.x = pack_i8x4(quant_i8(bf16_lo(u0.x), inv_sx0), quant_i8(bf16_hi(u0.x), inv_sx0), quant_i8(bf16_lo(u0.y), inv_sx0), quant_i8(bf16_hi(u0.y), inv_sx0));
              q.y = pack_i8x4(quant_i8(bf16_lo(u0.z), inv_sx0), quant_i8(bf16_hi(u0.z), inv_sx0), quant_i8(bf16_lo(u0.w), inv_sx0), quant_i8(bf16_hi(u0.w), inv_sx0));
              q.z = pack_i8x4(quant_i8(bf16_lo(u1.x), inv_sx0), quant_i8(bf16_hi(u1.x), inv_sx0), quant_i8(bf16_lo(u1.y), inv_sx0), quant_i8(bf16_hi(u1.y), inv_sx0));
              q.w = pack_i8x4(quant_i8(bf16_lo(u1.z), inv_sx0), quant_i8(bf16_hi(u1.z), inv_sx0), quant_i8(bf16_lo(u1.w), inv_sx0), quant_i8(bf16_hi(u1.w), inv_sx0));
            }
            *reinterpret_cast<uint4*>(blk + swz<KB>(r, piece)) = q;
          }
        } else {
          const float* base; int stride_el;                  // state rows are fp32: quantise while gathering
#pragma unroll
          for (int i = 0; i < CPR; ++i) {
            const int c = i * kUmmaThreads + tid, r = c / CPR, piece = c % CPR;
            size_t srow;
            if (KIND == kNodeNet) { base = static_cast<const float*>(s == 0 ? a.h : a.m); stride_el = s == 0 ? D : 2 * D; srow = (size_t)(row0 + r); }
            else if (s == 2) { base = static_cast<const float*>(a.e); stride_el = D; srow = (size_t)(row0 + r); }
            else { base = static_cast<const float*>(a.h); stride_el = D; srow = (size_t)IDX[s * kRows + r]; }
            const int col0 = (KIND == kNodeNet && s == 2) ? D : 0;
            uint4 q = make_uint4(0u, 0u, 0u, 0u);
            if (row0 + r < n_rows) {
              const float4* p = reinterpret_cast<const float4*>(base + srow * stride_el + col0 + piece * 16);
              const float4 f0 = __ldg(p), f1 = __ldg(p + 1), f2 = __ldg(p + 2), f3 = __ldg(p + 3);
              q.x = pack_i8x4(quant_i8(f0.x, inv_sx0), quant_i8(f0.y, inv_sx0), quant_i8(f0.z, inv_sx0), quant_i8(f0.w, inv_sx0));
              q.y = pack_i8x4(quant_i8(f1.x, inv_sx0), quant_i8(f1.y, inv_sx0), quant_i8(f1.z, inv_sx0), quant_i8(f1.w, inv_sx0));
              q.z = pack_i8x4(quant_i8(f2.x, inv_sx0), quant_i8(f2.y, inv_sx0), quant_i8(f2.z, inv_sx0), quant_i8(f2.w, inv_sx0));
              q.w = pack_i8x4(quant_i8(f3.x, inv_sx0), quant_i8(f3.y, inv_sx0), quant_i8(f3.z, inv_sx0), quant_i8(f3.w, inv_sx0));
            }
            *reinterpret_cast<uint4*>(blk + swz<KB>(r, piece)) = q;
          }
        }
      }
      fence_proxy_async();
      tc_fence_before();
      __syncthreads();
      // ---- layer 0 on the tensor cores: acc0 = A * W0^T ---------------------------------------------------------------
      if (warp == 0 && elect_one()) {
        tc_fence_after();
        issue_layer<PREC, KB>(a_addr, w0_addr, nseg * KB, D, tmem, idesc);
        umma_commit(bar_mma);
      }
      mbar_wait(bar_mma, phase); phase ^= 1;
      tc_fence_after();
      // ---- epilogue 0: bias, ReLU, operand conversion -> A tile of layer 1 ---------------------------------------------
      int32_t* tap_row = (PREC == kInt8 && a.tap && a.tap_layer == a.l0.index && live) ? a.tap + (size_t)row * D : nullptr;
#pragma unroll
      for (int c0 = 0; c0 < D; c0 += 32) {
        uint32_t v[32];
        tmem_ld32(tmem + lane_base + c0, v);
        store_hidden32<PREC, KB>(v, c0, scale0, bias0, inv_sx1, H, tid, tap_row);
      }
    } else {
      // ---- K = 3 input layer on the FFMA pipe (never a tensor layer, R20/R21), one row per thread ---------------
      float f0 = 0.f, f1 = 0.f, f2 = 0.f;
      if (live) {
        if (KIND == kNodeEnc) { const float4 f = a.feat[row]; f0 = f.x; f1 = f.y; f2 = f.z; }
        else {
          const float4 fs = a.feat[IDX[tid]], fd = a.feat[IDX[kRows + tid]];
          f0 = fabsf(__fsub_rn(fd.x, fs.x)); f1 = fabsf(__fsub_rn(fd.y, fs.y)); f2 = fabsf(__fsub_rn(fd.z, fs.z));
        }
      }
#pragma unroll
      for (int c0 = 0; c0 < D; c0 += 32) {
        float y[32];
#pragma unroll
        for (int j = 0; j < 32; ++j) {
          float acc = __fmaf_rn(f0, w3[c0 + j], 0.0f);
          acc = __fmaf_rn(f1, w3[D + c0 + j], acc);
          acc = __fmaf_rn(f2, w3[2 * D + c0 + j], acc);
          const float t = __fadd_rn(acc, bias0[c0 + j]);
          y[j] = t > 0.0f ? t : 0.0f;
        }
        store_operand32<PREC, KB>(y, c0, inv_sx1, H, tid);
      }
    }
    fence_proxy_async();
    tc_fence_before();
    __syncthreads();
    // ---- layer 1: acc1 = H * W1^T ---------------------------------------------------------------------------------------
    if (warp == 0 && elect_one()) {
      tc_fence_after();
      issue_layer<PREC, KB>(h_addr, w1_addr, KB, D, tmem + D, idesc);
      umma_commit(bar_mma);
    }
    mbar_wait(bar_mma, phase); phase ^= 1;
    tc_fence_after();
    // ---- epilogue 1: bias, residual, state store, optional edge classifier ---------------------------------------------
    {
      int32_t* tap_row = (PREC == kInt8 && a.tap && a.tap_layer == a.l1.index && live) ? a.tap + (size_t)row * D : nullptr;
      const bool residual = (KIND == kNodeNet || KIND == kEdgeNet);
      void* state = is_edge ? a.e : a.h;
      float hacc = 0.0f;
#pragma unroll
      for (int c0 = 0; c0 < D; c0 += 32) {
        uint32_t v[32];
        tmem_ld32(tmem + lane_base + D + c0, v);
        float y[32];
#pragma unroll
        for (int j = 0; j < 32; ++j) {
          const float acc = PREC == kBf16 ? __uint_as_float(v[j]) : (float)(int)v[j];
          y[j] = __fmaf_rn(acc, scale1[c0 + j], bias1[c0 + j]);
        }
        if (tap_row) {
#pragma unroll
          for (int j = 0; j < 32; ++j) tap_row[c0 + j] = (int)v[j];
        }
        if (live) {
          if (SB) {
            __nv_bfloat16* srow = static_cast<__nv_bfloat16*>(state) + (size_t)row * D + c0;
#pragma unroll
            for (int ch = 0; ch < 4; ++ch) {
              if (residual) {       // bf16 precision: the old state row is the e / h segment of the A tile (already in
                                    // shared memory); int8 precision: the A tile holds codes, re-read the row itself
                const int sseg = (KIND == kNodeNet) ? 0 : 2;
                const uint4 o = PREC == kBf16 ? *reinterpret_cast<const uint4*>(A + sseg * (kRows * KB) + swz<KB>(tid, (c0 * 2) / 16 + ch))
                                              : *reinterpret_cast<const uint4*>(srow + ch * 8);
                y[ch * 8 + 0] = __fadd_rn(bf16_lo(o.x), y[ch * 8 + 0]); y[ch * 8 + 1] = __fadd_rn(bf16_hi(o.x), y[ch * 8 + 1]);
                y[ch * 8 + 2] = __fadd_rn(bf16_lo(o.y), y[ch * 8 + 2]); y[ch * 8 + 3] = __fadd_rn(bf16_hi(o.y), y[ch * 8 + 3]);
                y[ch * 8 + 4] = __fadd_rn(bf16_lo(o.z), y[ch * 8 + 4]); y[ch * 8 + 5] = __fadd_rn(bf16_hi(o.z), y[ch * 8 + 5]);
                y[ch * 8 + 6] = __fadd_rn(bf16_lo(o.w), y[ch * 8 + 6]); y[ch * 8 + 7] = __fadd_rn(bf16_hi(o.w), y[ch * 8 + 7]);
              }
              uint4 q;
              q.x = pack_bf16x2(y[ch * 8 + 0], y[ch * 8 + 1]); q.y = pack_bf16x2(y[ch * 8 + 2], y[ch * 8 + 3]);
              q.z = pack_bf16x2(y[ch * 8 + 4], y[ch * 8 + 5]); q.w = pack_bf16x2(y[ch * 8 + 6], y[ch * 8 + 7]);
              *reinterpret_cast<uint4*>(srow + ch * 8) = q;
              if (is_edge && a.do_head) {      // the classifier sees the stored (bf16-rounded) state, R20
                y[ch * 8 + 0] = bf16_lo(q.x); y[ch * 8 + 1] = bf16_hi(q.x); y[ch * 8 + 2] = bf16_lo(q.y); y[ch * 8 + 3] = bf16_hi(q.y);
                y[ch * 8 + 4] = bf16_lo(q.z); y[ch * 8 + 5] = bf16_hi(q.z); y[ch * 8 + 6] = bf16_lo(q.w); y[ch * 8 + 7] = bf16_hi(q.w);
              }
            }
          } else {
            float* srow = static_cast<float*>(state) + (size_t)row * D + c0;
#pragma unroll
            for (int ch = 0; ch < 8; ++ch) {
              float4 o = make_float4(0.f, 0.f, 0.f, 0.f);
              if (residual) o = *reinterpret_cast<const float4*>(srow + ch * 4);
              if (residual) {
                y[ch * 4 + 0] = __fadd_rn(o.x, y[ch * 4 + 0]); y[ch * 4 + 1] = __fadd_rn(o.y, y[ch * 4 + 1]);
                y[ch * 4 + 2] = __fadd_rn(o.z, y[ch * 4 + 2]); y[ch * 4 + 3] = __fadd_rn(o.w, y[ch * 4 + 3]);
              }
              *reinterpret_cast<float4*>(srow + ch * 4) = make_float4(y[ch * 4 + 0], y[ch * 4 + 1], y[ch * 4 + 2], y[ch * 4 + 3]);
            }
          }
          if (is_edge && a.do_head) {
#pragma unroll
            for (int j = 0; j < 32; ++j) hacc = __fmaf_rn(y[j], headw[c0 + j], hacc);    // ascending j (R16)
          }
        }
      }
      if (is_edge && a.do_head && live) {
        const float z = __fadd_rn(hacc, head_b);
        a.logit[row] = z;
        a.score[row] = 1.0f / (1.0f + expf(-z));
      }
    }
    tc_fence_before();      // the next tile's MMAs overwrite the TMEM columns just read
  }
  __syncthreads();
  if (warp == 0) tmem_dealloc(tmem, TMEM_COLS);
}

// ============================================================================================================
// S1: embedding MLP 3 -> D -> ... -> D -> 4.  Layer 0 (K = 3) on the FFMA pipe, the D -> D layers
// and the D -> 4 output layer (N padded to 16) on the tensor cores; hidden activations never leave the SM.
struct UmmaEmbSmem { int a, w, par, bar, total; };
template <int PREC, int D>
__host__ __device__ constexpr UmmaEmbSmem emb_smem_layout(int n_mid) {
  constexpr int ESZ = PREC == kBf16 ? 2 : 1;
  UmmaEmbSmem s{};
  s.a = 0;                                            // activation tile [128][D*ESZ], overwritten in place per layer
  s.w = s.a + kRows * D * ESZ;                        // n_mid images [D][D*ESZ] + one [16][D*ESZ]
  s.par = s.w + n_mid * D * D * ESZ + 16 * D * ESZ;   // per tensor layer: scale[D], bias[D]; layer 0: W[3][D], b[D]
  s.bar = s.par + ((n_mid + 1) * 2 * D + 4 * D) * 4;
  s.total = s.bar + 32;
  return s;
}

template <int PREC, int D>
__global__ void __launch_bounds__(kUmmaThreads) embed_umma_kernel(EmbArgs a) {
  constexpr int ESZ = PREC == kBf16 ? 2 : 1;
  constexpr int ROWB = D * ESZ;                              // bytes per activation row
  constexpr int KB = ROWB > 128 ? 128 : ROWB;                // swizzle width
  constexpr uint32_t TMEM_COLS = 256;                        // hidden acc [0, D) | output acc [128, 144)
  const int H = a.n_layers - 1, n_mid = H - 1;               // tensor layers: n_mid (D -> D) + 1 (D -> 4)
  const UmmaEmbSmem L = emb_smem_layout<PREC, D>(n_mid);
  extern __shared__ uint8_t smem_raw[];
  uint8_t* smem = reinterpret_cast<uint8_t*>((reinterpret_cast<uintptr_t>(smem_raw) + 1023) & ~(uintptr_t)1023);
  uint8_t* A = smem + L.a; uint8_t* W = smem + L.w;
  float* par = reinterpret_cast<float*>(smem + L.par);
  float* w3 = par + (n_mid + 1) * 2 * D;                     // layer 0: W[3][D] then b[D]
  uint64_t* bar_w = reinterpret_cast<uint64_t*>(smem + L.bar);
  uint64_t* bar_mma = bar_w + 1;
  uint32_t* tmem_slot = reinterpret_cast<uint32_t*>(bar_w + 2);
  const int tid = threadIdx.x, warp = tid >> 5;

  if (tid == 0) { mbar_init(bar_w, 1); mbar_init(bar_mma, 1); fence_barrier_init(); }
  if (warp == 0) tmem_alloc(tmem_slot, TMEM_COLS);
  for (int l = 1; l <= H; ++l) {
    const LayerP& Ll = a.layers[l];
    for (int i = tid; i < D; i += kUmmaThreads) {
      par[(l - 1) * 2 * D + i] = i < Ll.N ? Ll.scale[i] : 0.0f;
      par[(l - 1) * 2 * D + D + i] = i < Ll.N ? Ll.bias[i] : 0.0f;
    }
  }
  for (int i = tid; i < D; i += kUmmaThreads) {
    w3[i] = a.layers[0].Wt[i]; w3[D + i] = a.layers[0].Wt[D + i]; w3[2 * D + i] = a.layers[0].Wt[2 * D + i];
    w3[3 * D + i] = a.layers[0].bias[i];
  }
  tc_fence_before();
  __syncthreads();
  tc_fence_after();
  const uint32_t tmem = *tmem_slot;
  if (tid == 0) {
    const uint32_t mid_bytes = (uint32_t)(D * ROWB), out_bytes = (uint32_t)(16 * ROWB);
    mbar_expect_tx(bar_w, n_mid * mid_bytes + out_bytes);
    for (int l = 0; l < n_mid; ++l) bulk_g2s(W + l * mid_bytes, a.layers[1 + l].Wtc, mid_bytes, bar_w);
    bulk_g2s(W + n_mid * mid_bytes, a.layers[H].Wtc, out_bytes, bar_w);
  }
  mbar_wait(bar_w, 0);
  const uint32_t a_addr = smem_u32(A), w_addr = smem_u32(W);
  const uint32_t lane_base = (uint32_t)(warp * 32) << 16;
  const uint32_t idesc_mid = make_idesc<PREC>(D), idesc_out = make_idesc<PREC>(16);
  uint32_t phase = 0;

  for (int tile = blockIdx.x; tile * kRows < a.n_rows; tile += gridDim.x) {
    const int row = tile * kRows + tid;
    const bool live = row < a.n_rows;
    __syncthreads();
    // ---- layer 0 (K = 3, FFMA): relu(W0 f + b0) -> operand of the first tensor layer ------------------------------
    {
      float4 f = live ? a.feat[row] : make_float4(0.f, 0.f, 0.f, 0.f);
      const float inv_next = a.layers[1].inv_sx;
#pragma unroll
      for (int c0 = 0; c0 < D; c0 += 32) {
        float y[32];
#pragma unroll
        for (int j = 0; j < 32; ++j) {
          float acc = __fmaf_rn(f.x, w3[c0 + j], 0.0f);
          acc = __fmaf_rn(f.y, w3[D + c0 + j], acc);
          acc = __fmaf_rn(f.z, w3[2 * D + c0 + j], acc);
          const float t = __fadd_rn(acc, w3[3 * D + c0 + j]);
          y[j] = t > 0.0f ? t : 0.0f;
        }
        store_operand32<PREC, KB>(y, c0, inv_next, A, tid);
      }
    }
    // ---- D -> D tensor layers, activation tile rewritten in place --------------------------------------------------
    for (int l = 0; l < n_mid; ++l) {
      fence_proxy_async();
      tc_fence_before();
      __syncthreads();
      if (warp == 0 && elect_one()) {
        tc_fence_after();
        issue_layer<PREC, KB>(a_addr, w_addr + l * (D * ROWB), ROWB, D, tmem, idesc_mid);
        umma_commit(bar_mma);
      }
      mbar_wait(bar_mma, phase); phase ^= 1;
      tc_fence_after();
      const LayerP& Ll = a.layers[1 + l];
      int32_t* tap_row = (PREC == kInt8 && a.tap && a.tap_layer == Ll.index && live) ? a.tap + (size_t)row * D : nullptr;
      const float inv_next = a.layers[2 + l].inv_sx;
#pragma unroll
      for (int c0 = 0; c0 < D; c0 += 32) {
        uint32_t v[32];
        tmem_ld32(tmem + lane_base + c0, v);
        store_hidden32<PREC, KB>(v, c0, par + l * 2 * D, par + l * 2 * D + D, inv_next, A, tid, tap_row);
      }
    }
    // ---- output layer D -> 4 (N padded to 16), linear, fp32 result (R20) -------------------------------------------
    fence_proxy_async();
    tc_fence_before();
    __syncthreads();
    if (warp == 0 && elect_one()) {
      tc_fence_after();
      issue_layer<PREC, KB>(a_addr, w_addr + n_mid * (D * ROWB), ROWB, 16, tmem + 128, idesc_out);
      umma_commit(bar_mma);
    }
    mbar_wait(bar_mma, phase); phase ^= 1;
    tc_fence_after();
    {
      uint32_t v[4];
      tmem_ld4(tmem + lane_base + 128, v);
      const float* sc = par + n_mid * 2 * D; const float* bi = sc + D;
      float y[4];
#pragma unroll
      for (int j = 0; j < 4; ++j) {
        const float acc = PREC == kBf16 ? __uint_as_float(v[j]) : (float)(int)v[j];
        y[j] = __fmaf_rn(acc, sc[j], bi[j]);
      }
      if (live) {
        a.emb[row] = make_float4(y[0], y[1], y[2], y[3]);
        if (PREC == kInt8 && a.tap && a.tap_layer == a.layers[H].index) {
#pragma unroll
          for (int j = 0; j < 4; ++j) a.tap[(size_t)row * 4 + j] = (int)v[j];
        }
      }
    }
    tc_fence_before();
  }
  __syncthreads();
  if (warp == 0) tmem_dealloc(tmem, TMEM_COLS);
}

// ---------------------------------------------------------------------------------------------- host side
// Shared-memory image of W[N][K] (K-major) as K-blocks of KB bytes with the UMMA swizzle applied, rows padded
// to n_pad.  `w` holds the operand values (bf16-representable floats or int8 codes) as [N][K] floats.
std::vector<uint8_t> pack_weight_image(const std::vector<float>& w, int N, int K, int n_pad, int esz, int KB) {
  const int rowb = K * esz, nkb = rowb / KB;
  std::vector<uint8_t> img((size_t)nkb * n_pad * KB, 0);
  for (int n = 0; n < N; ++n)
    for (int k = 0; k < K; ++k) {
      const int b = k * esz, kb = b / KB, within = b % KB, chunk = within / 16;
      const uint32_t lin = (uint32_t)n * KB;
      const size_t off = (size_t)kb * n_pad * KB + lin + (((chunk ^ (lin >> 7)) & (KB / 16 - 1)) << 4) + (within & 15);
      const float v = w[(size_t)n * K + k];
      if (esz == 2) {
        uint32_t u; memcpy(&u, &v, 4);
        img[off] = (uint8_t)((u >> 16) & 0xff); img[off + 1] = (uint8_t)(u >> 24);
      } else {
        img[off] = (uint8_t)(int8_t)(int)v;
      }
    }
  return img;
}

template <int KIND, int PREC, int D, bool SB>
void gnn_umma_launch_one(etx_ctx* c, const GnnArgs& a, int max_rows, cudaStream_t s) {
  auto kern = gnn_mlp_umma_kernel<KIND, PREC, D, SB>;
  constexpr int smem = gnn_smem_layout<PREC, D>().total + 1024;
  opt_in_smem(c, kern, smem);
  const int tiles = (max_rows + kRows - 1) / kRows;
  int per_sm = (227 * 1024) / (smem + 1024);
  const int tmem_cols = 2 * D < 32 ? 32 : 2 * D;
  if (per_sm > 512 / tmem_cols) per_sm = 512 / tmem_cols;
  if (per_sm < 1) per_sm = 1;
  const int grid = tiles < c->sm_count * per_sm ? tiles : c->sm_count * per_sm;
  if (grid <= 0) return;
  kern<<<grid, kUmmaThreads, smem, s>>>(a);
  c->launches++;
}

template <int PREC, int D, bool SB>
void gnn_umma_launch_kind(etx_ctx* c, int kind, const GnnArgs& a, int max_rows, cudaStream_t s) {
  switch (kind) {
    case kNodeEnc: gnn_umma_launch_one<kNodeEnc, PREC, D, SB>(c, a, max_rows, s); break;
    case kEdgeEnc: gnn_umma_launch_one<kEdgeEnc, PREC, D, SB>(c, a, max_rows, s); break;
    case kNodeNet: gnn_umma_launch_one<kNodeNet, PREC, D, SB>(c, a, max_rows, s); break;
    default:       gnn_umma_launch_one<kEdgeNet, PREC, D, SB>(c, a, max_rows, s); break;
  }
}

template <int PREC, int D>
void emb_umma_launch(etx_ctx* c, const EmbArgs& a, cudaStream_t s) {
  auto kern = embed_umma_kernel<PREC, D>;
  const int smem = emb_smem_layout<PREC, D>(a.n_layers - 2).total + 1024;
  opt_in_smem(c, kern, smem);
  const int tiles = (a.n_rows + kRows - 1) / kRows;
  int per_sm = (227 * 1024) / (smem + 1024);
  if (per_sm > 2) per_sm = 2;                               // 256 TMEM columns per CTA
  if (per_sm < 1) per_sm = 1;
  const int grid = tiles < c->sm_count * per_sm ? tiles : c->sm_count * per_sm;
  if (grid <= 0) return;
  kern<<<grid, kUmmaThreads, smem, s>>>(a);
  c->launches++;
}

}  // namespace

bool umma_supported(const etx_ctx* c) {
  if (c->precision != ETX_BF16 && c->precision != ETX_INT8) return false;
  const int D = c->hp.emb_hidden, d = c->hp.gnn_latent, H = c->hp.emb_n_hidden_layers;
  const int esz = c->precision == ETX_BF16 ? 2 : 1;
  const size_t emb_smem = (size_t)kRows * D * esz + (size_t)(H - 1) * D * D * esz + 16 * D * esz + 8192;
  return (D == 64 || D == 128) && (d == 32 || d == 64) && emb_smem <= 220 * 1024;
}

// pack every tensor layer's weights into its shared-memory image
void umma_configure(etx_ctx* c) {
  const int esz = c->precision == ETX_BF16 ? 2 : 1;
  for (auto& l : c->layers) {
    if (!l.tensor) continue;
    const bool is_emb = l.index < c->i_nenc;
    const int seg = is_emb ? l.in : c->hp.gnn_latent;        // K-block = one gathered segment (GNN) / 128 B (emb)
    int KB = seg * esz; if (KB > 128) KB = 128;
    const int n_pad = l.out < 16 ? 16 : l.out;
    std::vector<uint8_t> img = pack_weight_image(l.W, l.out, l.in, n_pad, esz, KB);
    void* p = etx_device_alloc(c, img.size());
    if (!p) { c->error = "device allocation (weight image)"; return; }
    cudaMemcpy(p, img.data(), img.size(), cudaMemcpyHostToDevice);
    l.dev.Wtc = p;
  }
}

void launch_embed_umma(etx_ctx* c, int n_hits, cudaStream_t s) {
  EmbArgs a;
  a.n_layers = c->hp.emb_n_hidden_layers + 1;
  for (int l = 0; l < a.n_layers; ++l) a.layers[l] = c->layers[c->i_emb0 + l].dev;
  a.feat = c->feat_emb; a.emb = c->emb; a.n_rows = n_hits;
  a.tap = c->tap_layer >= 0 ? c->tap : nullptr; a.tap_layer = c->tap_layer;
  const int D = c->hp.emb_hidden;
  if (c->precision == ETX_BF16) { if (D == 64) emb_umma_launch<kBf16, 64>(c, a, s); else emb_umma_launch<kBf16, 128>(c, a, s); }
  else { if (D == 64) emb_umma_launch<kInt8, 64>(c, a, s); else emb_umma_launch<kInt8, 128>(c, a, s); }
}

void launch_gnn_mlp_umma(etx_ctx* c, int kind, int iter, int n_hits, bool do_head, cudaStream_t s) {
  GnnArgs a;
  fill_gnn_args(c, kind, iter, n_hits, do_head, a);
  const bool is_edge = (kind == kEdgeEnc || kind == kEdgeNet);
  const long long max_rows_ll = is_edge ? (long long)n_hits * c->hp.k : n_hits;
  const int max_rows = (int)(max_rows_ll > 0x7fffffff ? 0x7fffffff : max_rows_ll);
  const int d = c->hp.gnn_latent;
  if (c->precision == ETX_BF16) { if (d == 32) gnn_umma_launch_kind<kBf16, 32, true>(c, kind, a, max_rows, s); else gnn_umma_launch_kind<kBf16, 64, true>(c, kind, a, max_rows, s); }
  else if (c->state_bf16) { if (d == 32) gnn_umma_launch_kind<kInt8, 32, true>(c, kind, a, max_rows, s); else gnn_umma_launch_kind<kInt8, 64, true>(c, kind, a, max_rows, s); }
  else { if (d == 32) gnn_umma_launch_kind<kInt8, 32, false>(c, kind, a, max_rows, s); else gnn_umma_launch_kind<kInt8, 64, false>(c, kind, a, max_rows, s); }
}

}  // namespace etx
