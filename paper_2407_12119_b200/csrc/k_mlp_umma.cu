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

#include "etx_internal.h"

namespace etx {

namespace {

enum { kBf16 = 0, kInt8 = 1 };
constexpr int kUmmaThreads = 128;   // 4 warps: warp w owns TMEM lanes 32w..32w+31 = rows 32w..32w+31
constexpr int kRows = 128;          // UMMA M

// ---------------------------------------------------------------------------------------------- PTX wrappers
__device__ __forceinline__ uint32_t smem_u32(const void* p) { return (uint32_t)__cvta_generic_to_shared(p); }

__device__ __forceinline__ void mbar_init(uint64_t* bar, uint32_t count) {
  asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(bar)), "r"(count) : "memory");
}
__device__ __forceinline__ void mbar_expect_tx(uint64_t* bar, uint32_t bytes) {
  asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(bar)), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_wait(uint64_t* bar, uint32_t parity) {
  const uint32_t addr = smem_u32(bar);
  uint32_t done = 0;
  for (uint32_t spins = 0; !done; ++spins) {
    asm volatile(
        "{\n\t.reg .pred p;\n\t"
        "mbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n\t"
        "selp.u32 %0, 1, 0, p;\n\t}"
        : "=r"(done) : "r"(addr), "r"(parity) : "memory");
    if (!done && spins > (1u << 24)) __trap();       // never hang the GPU: a lost arrival becomes an error
  }
}
__device__ __forceinline__ void fence_barrier_init() { asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory"); }
__device__ __forceinline__ void fence_proxy_async() { asm volatile("fence.proxy.async.shared::cta;" ::: "memory"); }
__device__ __forceinline__ void tc_fence_before() { asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory"); }
__device__ __forceinline__ void tc_fence_after() { asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory"); }

// TMA bulk copy global -> shared, completing on an mbarrier (SASS: UBLKCP)
__device__ __forceinline__ void bulk_g2s(void* dst, const void* src, uint32_t bytes, uint64_t* bar) {
  asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];"
               ::"r"(smem_u32(dst)), "l"(src), "r"(bytes), "r"(smem_u32(bar)) : "memory");
}

__device__ __forceinline__ void tmem_alloc(uint32_t* dst_smem, uint32_t cols) {   // one full warp
  asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], %1;" ::"r"(smem_u32(dst_smem)), "r"(cols) : "memory");
  asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;" ::: "memory");
}
__device__ __forceinline__ void tmem_dealloc(uint32_t taddr, uint32_t cols) {
  asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, %1;" ::"r"(taddr), "r"(cols) : "memory");
}

// D[tmem] (+)= A[smem] * B[smem]^T, M = 128, one thread issues
template <int PREC>
__device__ __forceinline__ void umma(uint32_t tmem_d, uint64_t adesc, uint64_t bdesc, uint32_t idesc, uint32_t accumulate) {
  if (PREC == kBf16)
    asm volatile("{\n\t.reg .pred p;\n\tsetp.ne.b32 p, %4, 0;\n\t"
                 "tcgen05.mma.cta_group::1.kind::f16 [%0], %1, %2, %3, p;\n\t}"
                 ::"r"(tmem_d), "l"(adesc), "l"(bdesc), "r"(idesc), "r"(accumulate) : "memory");
  else
    asm volatile("{\n\t.reg .pred p;\n\tsetp.ne.b32 p, %4, 0;\n\t"
                 "tcgen05.mma.cta_group::1.kind::i8 [%0], %1, %2, %3, p;\n\t}"
                 ::"r"(tmem_d), "l"(adesc), "l"(bdesc), "r"(idesc), "r"(accumulate) : "memory");
}
__device__ __forceinline__ void umma_commit(uint64_t* bar) {
  asm volatile("tcgen05.commit.cta_group::1.mbarrier::arrive::one.shared::cluster.b64 [%0];" ::"r"(smem_u32(bar)) : "memory");
}

// 32 lanes x 32 consecutive 32-bit columns: thread i of the warp gets lane (base + i)'s 32 columns
__device__ __forceinline__ void tmem_ld32(uint32_t taddr, uint32_t (&v)[32]) {
  asm volatile(
      "tcgen05.ld.sync.aligned.32x32b.x32.b32 "
      "{%0, %1, %2, %3, %4, %5, %6, %7, %8, %9, %10, %11, %12, %13, %14, %15, "
      "%16, %17, %18, %19, %20, %21, %22, %23, %24, %25, %26, %27, %28, %29, %30, %31}, [%32];"
      : "=r"(v[0]), "=r"(v[1]), "=r"(v[2]), "=r"(v[3]), "=r"(v[4]), "=r"(v[5]), "=r"(v[6]), "=r"(v[7]),
        "=r"(v[8]), "=r"(v[9]), "=r"(v[10]), "=r"(v[11]), "=r"(v[12]), "=r"(v[13]), "=r"(v[14]), "=r"(v[15]),
        "=r"(v[16]), "=r"(v[17]), "=r"(v[18]), "=r"(v[19]), "=r"(v[20]), "=r"(v[21]), "=r"(v[22]), "=r"(v[23]),
        "=r"(v[24]), "=r"(v[25]), "=r"(v[26]), "=r"(v[27]), "=r"(v[28]), "=r"(v[29]), "=r"(v[30]), "=r"(v[31])
      : "r"(taddr) : "memory");
  asm volatile("tcgen05.wait::ld.sync.aligned;" ::: "memory");
}
__device__ __forceinline__ void tmem_ld4(uint32_t taddr, uint32_t (&v)[4]) {
  asm volatile("tcgen05.ld.sync.aligned.32x32b.x4.b32 {%0, %1, %2, %3}, [%4];"
               : "=r"(v[0]), "=r"(v[1]), "=r"(v[2]), "=r"(v[3]) : "r"(taddr) : "memory");
  asm volatile("tcgen05.wait::ld.sync.aligned;" ::: "memory");
}

// ---------------------------------------------------------------------------------------------- descriptors
// K-major operand tile, swizzle width KB bytes: start address, LBO = 1 (unused for swizzled K-major),
// SBO = 8 rows * KB bytes, descriptor version 1 (sm_100), layout type 2 / 4 / 6 = SWIZZLE_128B / 64B / 32B.
template <int KB>
__device__ __forceinline__ uint64_t make_desc(uint32_t saddr) {
  constexpr uint64_t layout = KB == 128 ? 2 : (KB == 64 ? 4 : 6);
  uint64_t d = (uint64_t)((saddr & 0x3ffffu) >> 4);
  d |= (uint64_t)1 << 16;
  d |= (uint64_t)((8 * KB) >> 4) << 32;
  d |= (uint64_t)1 << 46;
  d |= layout << 61;
  return d;
}
// instruction descriptor: D fp32 / s32, A and B bf16 / s8, both K-major, N >> 3 at bit 17, M >> 4 at bit 24
template <int PREC>
__device__ __forceinline__ uint32_t make_idesc(int N) {
  const uint32_t fmt = PREC == kBf16 ? ((1u << 4) | (1u << 7) | (1u << 10)) : ((2u << 4) | (1u << 7) | (1u << 10));
  return fmt | ((uint32_t)(N >> 3) << 17) | ((uint32_t)(kRows >> 4) << 24);
}

// byte offset of 16-byte chunk `chunk` of row `r` inside a [rows][KB]-byte K-block
template <int KB>
__device__ __forceinline__ uint32_t swz(uint32_t r, uint32_t chunk) {
  const uint32_t lin = r * KB;
  return lin + (((chunk ^ (lin >> 7)) & (KB / 16 - 1)) << 4);
}

// issue all MMAs of one layer: K bytes of K extent (= K elements * esz), A/B as K-blocks of KB bytes
template <int PREC, int KB>
__device__ __forceinline__ void issue_layer(uint32_t a_base, uint32_t b_base, int kbytes, int n_rows_b, uint32_t tmem_d, uint32_t idesc) {
  const int steps = kbytes / 32;                          // 32 bytes of K per instruction (16 bf16 / 32 s8)
  for (int s = 0; s < steps; ++s) {
    const int kb = (s * 32) / KB, within = (s * 32) % KB;
    const uint64_t ad = make_desc<KB>(a_base + kb * (kRows * KB) + within);
    const uint64_t bd = make_desc<KB>(b_base + kb * (n_rows_b * KB) + within);
    umma<PREC>(tmem_d, ad, bd, idesc, s > 0 ? 1u : 0u);
  }
}

// ---------------------------------------------------------------------------------------------- conversions
__device__ __forceinline__ uint32_t pack_bf16x2(float lo, float hi) {       // RNE, lo in the low half
  uint32_t r;
  asm("cvt.rn.bf16x2.f32 %0, %1, %2;" : "=r"(r) : "f"(hi), "f"(lo));
  return r;
}
__device__ __forceinline__ float bf16_lo(uint32_t u) { return __uint_as_float(u << 16); }
__device__ __forceinline__ float bf16_hi(uint32_t u) { return __uint_as_float(u & 0xffff0000u); }
__device__ __forceinline__ int quant_i8(float x, float inv_s) {             // R21
  float r = rintf(__fmul_rn(x, inv_s));
  r = fminf(fmaxf(r, -127.0f), 127.0f);
  return __float2int_rn(r);
}
__device__ __forceinline__ uint32_t pack_i8x4(int a, int b, int c, int d) {
  return (uint32_t)(a & 0xff) | ((uint32_t)(b & 0xff) << 8) | ((uint32_t)(c & 0xff) << 16) | ((uint32_t)(d & 0xff) << 24);
}

// Row `r` of a K-major operand tile (K-blocks of KB bytes): store 32 consecutive hidden activations y (already
// biased and ReLU'd) starting at column c0, converted to the operand format: bf16 RNE (R20) or int8 codes (R21).
template <int PREC, int KB>
__device__ __forceinline__ void store_operand32(const float (&y)[32], int c0, float inv_sx_next, uint8_t* tile, uint32_t r) {
  constexpr int ESZ = PREC == kBf16 ? 2 : 1;
  constexpr int CH = 32 * ESZ / 16;                          // 16-byte chunks produced: 4 (bf16) or 2 (int8)
  const int byte0 = c0 * ESZ;
#pragma unroll
  for (int ch = 0; ch < CH; ++ch) {
    uint4 q;
    if (PREC == kBf16) {
      q.x = pack_bf16x2(y[ch * 8 + 0], y[ch * 8 + 1]); q.y = pack_bf16x2(y[ch * 8 + 2], y[ch * 8 + 3]);
      q.z = pack_bf16x2(y[ch * 8 + 4], y[ch * 8 + 5]); q.w = pack_bf16x2(y[ch * 8 + 6], y[ch * 8 + 7]);
    } else {
      int t[16];
#pragma unroll
      for (int j = 0; j < 16; ++j) t[j] = quant_i8(y[ch * 16 + j], inv_sx_next);
      q.x = pack_i8x4(t[0], t[1], t[2], t[3]); q.y = pack_i8x4(t[4], t[5], t[6], t[7]);
      q.z = pack_i8x4(t[8], t[9], t[10], t[11]); q.w = pack_i8x4(t[12], t[13], t[14], t[15]);
    }
    const int b = byte0 + ch * 16;
    const int kb = b / KB, chunk = (b % KB) / 16;
    *reinterpret_cast<uint4*>(tile + kb * (kRows * KB) + swz<KB>(r, chunk)) = q;
  }
}

// epilogue of a hidden tensor layer: y = relu(fmaf(acc, scale, bias)) on 32 accumulator columns, then store
template <int PREC, int KB>
__device__ __forceinline__ void store_hidden32(const uint32_t (&v)[32], int c0, const float* __restrict__ scale,
                                               const float* __restrict__ bias, float inv_sx_next, uint8_t* tile, uint32_t r,
                                               int32_t* tap_row) {
  float y[32];
#pragma unroll
  for (int j = 0; j < 32; ++j) {
    const float acc = PREC == kBf16 ? __uint_as_float(v[j]) : (float)(int)v[j];
    const float t = __fmaf_rn(acc, scale[c0 + j], bias[c0 + j]);
    y[j] = t > 0.0f ? t : 0.0f;
  }
  if (PREC == kInt8 && tap_row) {
#pragma unroll
    for (int j = 0; j < 32; ++j) tap_row[c0 + j] = (int)v[j];
  }
  store_operand32<PREC, KB>(y, c0, inv_sx_next, tile, r);
}

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

template <int KIND, int PREC, int D>
__global__ void __launch_bounds__(kUmmaThreads) gnn_mlp_umma_kernel(GnnArgs a) {
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
      if (tid == 0) {
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
    if (tid == 0) {
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
          if (PREC == kBf16) {
            __nv_bfloat16* srow = static_cast<__nv_bfloat16*>(state) + (size_t)row * D + c0;
#pragma unroll
            for (int ch = 0; ch < 4; ++ch) {
              if (residual) {       // the old state row is the e / h segment of the A tile (already in shared memory)
                const int sseg = (KIND == kNodeNet) ? 0 : 2;
                const uint4 o = *reinterpret_cast<const uint4*>(A + sseg * (kRows * KB) + swz<KB>(tid, (c0 * 2) / 16 + ch));
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
      if (tid == 0) {
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
    if (tid == 0) {
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

template <int KIND, int PREC, int D>
void gnn_umma_launch_one(etx_ctx* c, const GnnArgs& a, int max_rows, cudaStream_t s) {
  auto kern = gnn_mlp_umma_kernel<KIND, PREC, D>;
  constexpr int smem = gnn_smem_layout<PREC, D>().total + 1024;
  static bool configured = false;
  if (!configured) { cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, smem); configured = true; }
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

template <int PREC, int D>
void gnn_umma_launch_kind(etx_ctx* c, int kind, const GnnArgs& a, int max_rows, cudaStream_t s) {
  switch (kind) {
    case kNodeEnc: gnn_umma_launch_one<kNodeEnc, PREC, D>(c, a, max_rows, s); break;
    case kEdgeEnc: gnn_umma_launch_one<kEdgeEnc, PREC, D>(c, a, max_rows, s); break;
    case kNodeNet: gnn_umma_launch_one<kNodeNet, PREC, D>(c, a, max_rows, s); break;
    default:       gnn_umma_launch_one<kEdgeNet, PREC, D>(c, a, max_rows, s); break;
  }
}

template <int PREC, int D>
void emb_umma_launch(etx_ctx* c, const EmbArgs& a, cudaStream_t s) {
  auto kern = embed_umma_kernel<PREC, D>;
  const int smem = emb_smem_layout<PREC, D>(a.n_layers - 2).total + 1024;
  cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, smem);
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
    void* p = nullptr;
    if (cudaMalloc(&p, img.size()) != cudaSuccess) { c->error = "cudaMalloc(weight image)"; return; }
    c->allocs.push_back(p);
    cudaMemcpy(p, img.data(), img.size(), cudaMemcpyHostToDevice);
    l.dev.Wtc = p;
  }
}

void launch_embed_umma(etx_ctx* c, int n_hits, cudaStream_t s) {
  EmbArgs a;
  a.n_layers = c->hp.emb_n_hidden_layers + 1;
  for (int l = 0; l < a.n_layers; ++l) a.layers[l] = c->layers[c->i_emb0 + l].dev;
  a.feat = c->feat; a.emb = c->emb; a.n_rows = n_hits;
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
  if (c->precision == ETX_BF16) { if (d == 32) gnn_umma_launch_kind<kBf16, 32>(c, kind, a, max_rows, s); else gnn_umma_launch_kind<kBf16, 64>(c, kind, a, max_rows, s); }
  else { if (d == 32) gnn_umma_launch_kind<kInt8, 32>(c, kind, a, max_rows, s); else gnn_umma_launch_kind<kInt8, 64>(c, kind, a, max_rows, s); }
}

}  // namespace etx
