// S4e, INT8 mode (R21): e <- e + MLP_k([h_src, h_dst, e]) with int8 operands, int32 accumulation on
// tcgen05 (kind::i8), fp32 dequantisation + bias + ReLU, fp32 state.  PAPER.md L140, L148; the paper quantised only
// its embedding (L265-269) and names the GNN as the step where INT8 would pay most (L271).
//
// Same arithmetic, operation for operation, as gnn_mlp_umma_kernel<kEdgeNet, kInt8, D> (every int32 accumulator is
// reproduced bit for bit, and every other op is a single pinned fp32 op), but warp-specialised and pipelined, with
// the fp32 edge state moved by TMA as in the bf16 kernel (k_edge_tma.cu):
//
//   TMA loader (1 thread) the 128-row fp32 tile of e (contiguous) -> a 128B-swizzled slot of a kI8E-deep ring;
//   producers  (8 warps)  gather the fp32 rows h[src] | h[dst] from global memory (L2 hits), take e from the slot,
//                         quantise all three (q = clamp(rne(x * (1 / s_x)), +-127)) into the int8 A tile;
//   MMA issuer (1 thread) layer 0 of tile i+1 is issued before layer 1 of tile i; accumulators double-buffered in TMEM;
//   epilogue   (2 x 4 warps) warpgroup g owns tiles i = g (mod 2): acc0 -> fmaf(acc, s_x s_w, b) -> relu -> int8 ->
//                         layer-1 operand; acc1 -> fmaf -> + old e, IN PLACE in the slot, and the classifier dot
//                         product on the last step;
//   TMA storer (1 thread) the slot -> e, then hands the slot back to the loader.
#include <cuda.h>
#include <string.h>

#include "umma_common.cuh"

namespace etx {

namespace {

using namespace umma;

constexpr int kI8E = 4;                                    // ring of fp32 edge-state tiles (6 when the state is bf16: half the bytes per tile)
constexpr int kI8A = 2;                                    // ring of int8 operand tiles
constexpr int kI8EpiWarps = 8, kI8ProdWarps = 8;
constexpr int kI8MmaWarp = kI8EpiWarps + kI8ProdWarps, kI8LoadWarp = kI8MmaWarp + 1, kI8StoreWarp = kI8MmaWarp + 2;
constexpr int kI8Threads = (kI8StoreWarp + 1) * 32;        // 608
constexpr int kI8ProdThreads = kI8ProdWarps * 32;
// ptxas compiles the 608-thread CTA with 96 registers per thread; the two producer warpgroups hand 16 each to the
// two epilogue warpgroups: 256 * 80 + 256 * 112 + 96 * 96 = 58368 = 608 * 96.
constexpr int kI8ProdRegs = 80, kI8EpiRegs = 112;
constexpr int kI8Sub = kRows * 128;                        // one TMA box of the fp32 tile: [128 rows][32 floats]

__device__ __forceinline__ void tma_load_2d(uint32_t dst, const CUtensorMap* map, int x, int y, uint64_t* bar) {
  asm volatile("cp.async.bulk.tensor.2d.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1, {%3, %4}], [%2];"
               ::"r"(dst), "l"(reinterpret_cast<uint64_t>(map)), "r"(smem_u32(bar)), "r"(x), "r"(y) : "memory");
}
__device__ __forceinline__ void tma_store_2d(const CUtensorMap* map, uint32_t src, int x, int y) {
  asm volatile("cp.async.bulk.tensor.2d.global.shared::cta.bulk_group [%0, {%2, %3}], [%1];"
               ::"l"(reinterpret_cast<uint64_t>(map)), "r"(src), "r"(x), "r"(y) : "memory");
}

// byte offset of floats [4 c4, 4 c4 + 4) of row r inside an fp32 tile slot (boxes of 32 floats, 128B swizzle)
__device__ __forceinline__ uint32_t e_off(uint32_t r, uint32_t c4) {
  return (c4 >> 3) * kI8Sub + r * 128 + (((c4 & 7) ^ (r & 7)) << 4);
}

struct I8Smem { int e, a, h, w0, w1, par, bar, total; };
template <int D, bool SB>
__host__ __device__ constexpr I8Smem i8_layout() {
  I8Smem s{};
  s.e = 0;                                   // NE x [128][D] state tile: fp32 as D/32 boxes [128][128 B], bf16 as one box [128][2 D B]
  s.a = s.e + (SB ? 6 : kI8E) * kRows * D * (SB ? 2 : 4);   // kI8A x 3 K-blocks [128][D] int8
  s.h = s.a + kI8A * 3 * kRows * D;          // 2 x [128][D]: layer-1 operand per epilogue warpgroup
  s.w0 = s.h + 2 * kRows * D;                // W0 image: 3 K-blocks [D][D]
  s.w1 = s.w0 + 3 * D * D;                   // W1 image
  s.par = s.w1 + D * D;                      // fp32: scale0, bias0, scale1, bias1, head w
  s.bar = s.par + 5 * D * 4;
  s.total = s.bar + 256;
  return s;
}

// NODE = false: S4e over edges (self state e, K-block 2; gathered h[src], h[dst]);  NODE = true: S4d over hits
// (self state h, K-block 0; m_out, m_in of the same row).
// SB: the state rows (h, e, m) are bf16 (state_dtype = bf16, R21): one TMA box per tile, half the bytes, a deeper ring;
// values are widened to fp32 before every arithmetic step and rounded (RNE) only when the new state is stored.
template <int D, bool NODE, bool SB>
__global__ void __launch_bounds__(kI8Threads, 1) edge_net_i8_kernel(const __grid_constant__ CUtensorMap e_map, GnnArgs a) {
  constexpr int KB = D;                                      // bytes per int8 segment row = swizzle width (32 / 64)
  constexpr int CPR = KB / 16;                               // 16-byte chunks per segment row
  constexpr int BLK = kRows * KB;
  constexpr int STAGE = 3 * BLK;
  constexpr int NE = SB ? 6 : kI8E;                          // depth of the state ring
  constexpr int SROW = D * (SB ? 2 : 4);                     // bytes per state row
  constexpr int ETILE = kRows * SROW;
  constexpr I8Smem L = i8_layout<D, SB>();
  constexpr uint32_t TMEM_COLS = 4 * D;                      // acc0[2] | acc1[2]
  extern __shared__ uint8_t smem_raw[];
  uint8_t* smem = reinterpret_cast<uint8_t*>((reinterpret_cast<uintptr_t>(smem_raw) + 1023) & ~(uintptr_t)1023);
  float* par = reinterpret_cast<float*>(smem + L.par);
  float *scale0 = par, *bias0 = par + D, *scale1 = par + 2 * D, *bias1 = par + 3 * D, *headw = par + 4 * D;
  uint64_t* bars = reinterpret_cast<uint64_t*>(smem + L.bar);
  uint64_t *e_full = bars, *e_free = bars + NE, *out_ready = bars + 2 * NE, *a_full = bars + 3 * NE,
           *a_empty = a_full + kI8A, *acc0_full = a_empty + kI8A, *hid_full = acc0_full + 2, *acc1_full = acc0_full + 4,
           *bar_w = acc0_full + 6;
  uint32_t* tmem_slot = reinterpret_cast<uint32_t*>(acc0_full + 7);

  const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
  const int n_rows = NODE ? a.n_rows : *a.n_rows_ptr;
  const int n_tiles = (n_rows + kRows - 1) / kRows;
  constexpr int SELF = NODE ? 0 : 2, AUX0 = NODE ? 1 : 0, AUX1 = NODE ? 2 : 1;   // K-blocks of the A tile

  if (tid == 0) {
    for (int s = 0; s < NE; ++s) { mbar_init(&e_full[s], 1); mbar_init(&e_free[s], 1); mbar_init(&out_ready[s], 128); }
    for (int s = 0; s < kI8A; ++s) { mbar_init(&a_full[s], kI8ProdThreads); mbar_init(&a_empty[s], 1); }
    for (int g = 0; g < 2; ++g) { mbar_init(&acc0_full[g], 1); mbar_init(&hid_full[g], 128); mbar_init(&acc1_full[g], 1); }
    mbar_init(bar_w, 1);
    fence_barrier_init();
  }
  if (warp == kI8MmaWarp) tmem_alloc(tmem_slot, TMEM_COLS);
  for (int i = tid; i < D; i += kI8Threads) {
    scale0[i] = a.l0.scale[i]; bias0[i] = a.l0.bias[i]; scale1[i] = a.l1.scale[i]; bias1[i] = a.l1.bias[i];
    headw[i] = a.head.Wt[i];
  }
  tc_fence_before();
  __syncthreads();
  tc_fence_after();
  const uint32_t tmem = *tmem_slot;
  const uint32_t e_addr = smem_u32(smem + L.e);

  if (warp >= kI8EpiWarps && warp < kI8MmaWarp) {
    // ================================================================================================ producers
    asm volatile("setmaxnreg.dec.sync.aligned.u32 %0;" ::"n"(kI8ProdRegs));
    const int pt = tid - kI8EpiWarps * 32;                   // 0 .. 255
    const float inv_sx0 = a.l0.inv_sx;
    const float* hbase = static_cast<const float*>(a.h);
    const __nv_bfloat16* hbase16 = static_cast<const __nv_bfloat16*>(a.h);
    auto quant16 = [&](const float4& f0, const float4& f1, const float4& f2, const float4& f3) {
      uint4 q;
      q.x = pack_i8x4(quant_i8(f0.x, inv_sx0), quant_i8(f0.y, inv_sx0), quant_i8(f0.z, inv_sx0), quant_i8(f0.w, inv_sx0));
      q.y = pack_i8x4(quant_i8(f1.x, inv_sx0), quant_i8(f1.y, inv_sx0), quant_i8(f1.z, inv_sx0), quant_i8(f1.w, inv_sx0));
      q.z = pack_i8x4(quant_i8(f2.x, inv_sx0), quant_i8(f2.y, inv_sx0), quant_i8(f2.z, inv_sx0), quant_i8(f2.w, inv_sx0));
      q.w = pack_i8x4(quant_i8(f3.x, inv_sx0), quant_i8(f3.y, inv_sx0), quant_i8(f3.z, inv_sx0), quant_i8(f3.w, inv_sx0));
      return q;
    };
    auto quant16b = [&](const uint4& u0, const uint4& u1) {     // 16 bf16 values, widened exactly
      uint4 q;
      q.x = pack_i8x4(quant_i8(bf16_lo(u0.x), inv_sx0), quant_i8(bf16_hi(u0.x), inv_sx0), quant_i8(bf16_lo(u0.y), inv_sx0), quant_i8(bf16_hi(u0.y), inv_sx0));
      q.y = pack_i8x4(quant_i8(bf16_lo(u0.z), inv_sx0), quant_i8(bf16_hi(u0.z), inv_sx0), quant_i8(bf16_lo(u0.w), inv_sx0), quant_i8(bf16_hi(u0.w), inv_sx0));
      q.z = pack_i8x4(quant_i8(bf16_lo(u1.x), inv_sx0), quant_i8(bf16_hi(u1.x), inv_sx0), quant_i8(bf16_lo(u1.y), inv_sx0), quant_i8(bf16_hi(u1.y), inv_sx0));
      q.w = pack_i8x4(quant_i8(bf16_lo(u1.z), inv_sx0), quant_i8(bf16_hi(u1.z), inv_sx0), quant_i8(bf16_lo(u1.w), inv_sx0), quant_i8(bf16_hi(u1.w), inv_sx0));
      return q;
    };
    int it = 0;
    if (!NODE && a.hq_in != nullptr) {
      // h[src], h[dst] arrive as int8 codes (written by the node network under this layer's input scale): the producers
      // only move them.  The gather is a dependent chain (index -> code row) of L2 round trips, so it is software-
      // pipelined in registers: codes one tile ahead, indices two tiles ahead; the only values quantised here are the
      // tile's own state rows.
      constexpr int ITEMS = (kRows * CPR + kI8ProdThreads - 1) / kI8ProdThreads;
      auto load_idx = [&](long long tile, int (&js)[ITEMS], int (&jd)[ITEMS]) {
#pragma unroll
        for (int i = 0; i < ITEMS; ++i) {
          const int c = i * kI8ProdThreads + pt;
          js[i] = 0; jd[i] = 0;
          if (tile < n_tiles && c < kRows * CPR) {
            long long grow = tile * kRows + c / CPR;
            if (grow >= n_rows) grow = n_rows - 1;
            js[i] = __ldg(a.src + grow); jd[i] = __ldg(a.dst + grow);
          }
        }
      };
      auto load_codes = [&](const int (&js)[ITEMS], const int (&jd)[ITEMS], uint4 (&cs)[ITEMS], uint4 (&cd)[ITEMS]) {
#pragma unroll
        for (int i = 0; i < ITEMS; ++i) {
          const int piece = (i * kI8ProdThreads + pt) % CPR;
          cs[i] = __ldg(reinterpret_cast<const uint4*>(a.hq_in + (size_t)js[i] * D) + piece);
          cd[i] = __ldg(reinterpret_cast<const uint4*>(a.hq_in + (size_t)jd[i] * D) + piece);
        }
      };
      int js1[ITEMS], jd1[ITEMS], js2[ITEMS], jd2[ITEMS];
      uint4 cs0[ITEMS], cd0[ITEMS], cs1[ITEMS], cd1[ITEMS];
      load_idx(blockIdx.x, js1, jd1);
      load_codes(js1, jd1, cs0, cd0);                                // codes of the first tile
      load_idx((long long)blockIdx.x + gridDim.x, js1, jd1);         // indices of the second
      for (long long tile = blockIdx.x; tile < n_tiles; tile += gridDim.x, ++it) {
        const int sa = it % kI8A, se = it % NE;
        uint8_t* st = smem + L.a + sa * STAGE;
        const uint8_t* es = smem + L.e + se * ETILE;
        if (tile + gridDim.x < n_tiles) load_codes(js1, jd1, cs1, cd1);   // next tile's codes: in flight under this tile
        load_idx(tile + 2LL * gridDim.x, js2, jd2);
        mbar_wait(&a_empty[sa], ((it / kI8A) & 1) ^ 1);
        mbar_wait(&e_full[se], (it / NE) & 1);
#pragma unroll
        for (int i = 0; i < ITEMS; ++i) {
          const int c = i * kI8ProdThreads + pt;
          if (c < kRows * CPR) {
            const int r = c / CPR, piece = c % CPR;
            uint4 q;
            if (SB) {
              const uint4 e0 = *reinterpret_cast<const uint4*>(es + swz<SROW>(r, piece * 2 + 0));
              const uint4 e1 = *reinterpret_cast<const uint4*>(es + swz<SROW>(r, piece * 2 + 1));
              q = quant16b(e0, e1);
            } else {
              const float4 e0 = *reinterpret_cast<const float4*>(es + e_off(r, piece * 4 + 0));
              const float4 e1 = *reinterpret_cast<const float4*>(es + e_off(r, piece * 4 + 1));
              const float4 e2 = *reinterpret_cast<const float4*>(es + e_off(r, piece * 4 + 2));
              const float4 e3 = *reinterpret_cast<const float4*>(es + e_off(r, piece * 4 + 3));
              q = quant16(e0, e1, e2, e3);
            }
            *reinterpret_cast<uint4*>(st + SELF * BLK + swz<KB>(r, piece)) = q;
            *reinterpret_cast<uint4*>(st + AUX0 * BLK + swz<KB>(r, piece)) = cs0[i];
            *reinterpret_cast<uint4*>(st + AUX1 * BLK + swz<KB>(r, piece)) = cd0[i];
          }
        }
        fence_proxy_async();                                    // generic-proxy writes -> visible to the tensor core
        mbar_arrive(&a_full[sa]);
#pragma unroll
        for (int i = 0; i < ITEMS; ++i) { cs0[i] = cs1[i]; cd0[i] = cd1[i]; js1[i] = js2[i]; jd1[i] = jd2[i]; }
      }
    } else
    for (int tile = blockIdx.x; tile < n_tiles; tile += gridDim.x, ++it) {
      const int sa = it % kI8A, se = it % NE;
      uint8_t* st = smem + L.a + sa * STAGE;
      const uint8_t* es = smem + L.e + se * ETILE;
      bool first = true;
      // item c = (row r, 16-byte chunk `piece` of the int8 row) = 16 consecutive values of the source row
#pragma unroll
      for (int i = 0; i < (kRows * CPR + kI8ProdThreads - 1) / kI8ProdThreads; ++i) {
        const int c = i * kI8ProdThreads + pt;
        if (c < kRows * CPR) {
          const int r = c / CPR, piece = c % CPR;
          int grow = tile * kRows + r;
          if (grow >= n_rows) grow = n_rows - 1;              // dead rows of the last tile: any valid row (never stored)
          if (SB) {
            const uint4 *ps, *pd;
            if (NODE) {
              ps = reinterpret_cast<const uint4*>(static_cast<const __nv_bfloat16*>(a.m) + (size_t)grow * 2 * D + piece * 16);
              pd = ps + D / 8;
            } else {
              const int js = __ldg(a.src + grow), jd = __ldg(a.dst + grow);
              ps = reinterpret_cast<const uint4*>(hbase16 + (size_t)js * D + piece * 16);
              pd = reinterpret_cast<const uint4*>(hbase16 + (size_t)jd * D + piece * 16);
            }
            const uint4 s0 = __ldg(ps), s1 = __ldg(ps + 1), d0 = __ldg(pd), d1 = __ldg(pd + 1);
            if (first) {                                      // the gathers are in flight while we wait for the slots
              mbar_wait(&a_empty[sa], ((it / kI8A) & 1) ^ 1);
              mbar_wait(&e_full[se], (it / NE) & 1);
              first = false;
            }
            const uint4 e0 = *reinterpret_cast<const uint4*>(es + swz<SROW>(r, piece * 2 + 0));
            const uint4 e1 = *reinterpret_cast<const uint4*>(es + swz<SROW>(r, piece * 2 + 1));
            *reinterpret_cast<uint4*>(st + SELF * BLK + swz<KB>(r, piece)) = quant16b(e0, e1);
            *reinterpret_cast<uint4*>(st + AUX0 * BLK + swz<KB>(r, piece)) = quant16b(s0, s1);
            *reinterpret_cast<uint4*>(st + AUX1 * BLK + swz<KB>(r, piece)) = quant16b(d0, d1);
          } else {
          const float4 *ps, *pd;
          if (NODE) {
            ps = reinterpret_cast<const float4*>(static_cast<const float*>(a.m) + (size_t)grow * 2 * D + piece * 16);
            pd = ps + D / 4;
          } else {
            const int js = __ldg(a.src + grow), jd = __ldg(a.dst + grow);
            ps = reinterpret_cast<const float4*>(hbase + (size_t)js * D + piece * 16);
            pd = reinterpret_cast<const float4*>(hbase + (size_t)jd * D + piece * 16);
          }
          const float4 s0 = __ldg(ps), s1 = __ldg(ps + 1), s2 = __ldg(ps + 2), s3 = __ldg(ps + 3);
          const float4 d0 = __ldg(pd), d1 = __ldg(pd + 1), d2 = __ldg(pd + 2), d3 = __ldg(pd + 3);
          if (first) {                                        // the gathers are in flight while we wait for the slots
            mbar_wait(&a_empty[sa], ((it / kI8A) & 1) ^ 1);
            mbar_wait(&e_full[se], (it / NE) & 1);
            first = false;
          }
          const float4 e0 = *reinterpret_cast<const float4*>(es + e_off(r, piece * 4 + 0));
          const float4 e1 = *reinterpret_cast<const float4*>(es + e_off(r, piece * 4 + 1));
          const float4 e2 = *reinterpret_cast<const float4*>(es + e_off(r, piece * 4 + 2));
          const float4 e3 = *reinterpret_cast<const float4*>(es + e_off(r, piece * 4 + 3));
          *reinterpret_cast<uint4*>(st + SELF * BLK + swz<KB>(r, piece)) = quant16(e0, e1, e2, e3);
          *reinterpret_cast<uint4*>(st + AUX0 * BLK + swz<KB>(r, piece)) = quant16(s0, s1, s2, s3);
          *reinterpret_cast<uint4*>(st + AUX1 * BLK + swz<KB>(r, piece)) = quant16(d0, d1, d2, d3);
          }
        }
      }
      if (first) { mbar_wait(&a_empty[sa], ((it / kI8A) & 1) ^ 1); mbar_wait(&e_full[se], (it / NE) & 1); }
      fence_proxy_async();                                    // generic-proxy writes -> visible to the tensor core
      mbar_arrive(&a_full[sa]);
    }
  } else if (warp == kI8LoadWarp) {
    // ================================================================================================ TMA loads
    if (lane == 0) {
      int it = 0;
      for (int tile = blockIdx.x; tile < n_tiles; tile += gridDim.x, ++it) {
        const int s = it % NE;
        mbar_wait(&e_free[s], ((it / NE) & 1) ^ 1);
        mbar_expect_tx(&e_full[s], ETILE);
        if (SB) tma_load_2d(e_addr + s * ETILE, &e_map, 0, tile * kRows, &e_full[s]);
        else {
#pragma unroll
          for (int b = 0; b < D / 32; ++b) tma_load_2d(e_addr + s * ETILE + b * kI8Sub, &e_map, 32 * b, tile * kRows, &e_full[s]);
        }
      }
    }
  } else if (warp == kI8StoreWarp) {
    // ================================================================================================ TMA stores
    if (lane == 0) {
      int it = 0;
      for (int tile = blockIdx.x; tile < n_tiles; tile += gridDim.x, ++it) {
        const int s = it % NE;
        mbar_wait(&out_ready[s], (it / NE) & 1);
        if (a.do_head != 2) {                                 // 2: the new state is dead (last step of a plain etx_run)
          if (SB) tma_store_2d(&e_map, e_addr + s * ETILE, 0, tile * kRows);
          else {
#pragma unroll
            for (int b = 0; b < D / 32; ++b) tma_store_2d(&e_map, e_addr + s * ETILE + b * kI8Sub, 32 * b, tile * kRows);
          }
          asm volatile("cp.async.bulk.commit_group;" ::: "memory");
          asm volatile("cp.async.bulk.wait_group.read 0;" ::: "memory");
        }
        mbar_arrive(&e_free[s]);
      }
      asm volatile("cp.async.bulk.wait_group 0;" ::: "memory");
    }
  } else if (warp == kI8MmaWarp) {
    // ================================================================================================ MMA issuer
    if (elect_one()) {
      const uint32_t b0 = (uint32_t)(3 * D * KB), b1 = (uint32_t)(D * KB);
      mbar_expect_tx(bar_w, b0 + b1);
      bulk_g2s(smem + L.w0, a.l0.Wtc, b0, bar_w);
      bulk_g2s(smem + L.w1, a.l1.Wtc, b1, bar_w);
      mbar_wait(bar_w, 0);
      const uint32_t idesc = make_idesc<kInt8>(D);
      const uint32_t a_addr = smem_u32(smem + L.a), h_addr = smem_u32(smem + L.h);
      const uint32_t w0_addr = smem_u32(smem + L.w0), w1_addr = smem_u32(smem + L.w1);
      auto layer1 = [&](int j) {                              // layer 1 of the CTA's j-th tile
        const int g = j & 1;
        mbar_wait(&hid_full[g], (j >> 1) & 1);
        tc_fence_after();
        issue_layer<kInt8, KB>(h_addr + g * BLK, w1_addr, KB, D, tmem + 2 * D + g * D, idesc);
        umma_commit(&acc1_full[g]);
      };
      int it = 0;
      for (int tile = blockIdx.x; tile < n_tiles; tile += gridDim.x, ++it) {
        const int s = it % kI8A, g = it & 1;
        mbar_wait(&a_full[s], (it / kI8A) & 1);
        tc_fence_after();
        // acc0[g] was drained by epilogue 0 of tile it-2, which hid_full (waited on for layer 1 of it-2) covers
        issue_layer<kInt8, KB>(a_addr + s * STAGE, w0_addr, 3 * KB, D, tmem + g * D, idesc);
        umma_commit(&acc0_full[g]);
        umma_commit(&a_empty[s]);                             // layer 0 is the operand tile's only reader
        if (it > 0) layer1(it - 1);
      }
      if (it > 0) layer1(it - 1);
    }
  } else {
    // ================================================================================================ epilogue
    asm volatile("setmaxnreg.inc.sync.aligned.u32 %0;" ::"n"(kI8EpiRegs));
    const int g = warp >> 2, q = warp & 3;                    // warpgroup, TMEM lane quarter
    const int r = q * 32 + lane;                              // row of the tile owned by this thread
    const uint32_t lane_base = (uint32_t)(q * 32) << 16;
    uint8_t* Hg = smem + L.h + g * BLK;
    const float head_b = a.head.bias[0];
    const float inv_sx1 = a.l1.inv_sx;
    int j = 0;                                                // this warpgroup's tile counter
    for (int it = g; blockIdx.x + (long long)it * gridDim.x < n_tiles; it += 2, ++j) {
      const long long tile = blockIdx.x + (long long)it * gridDim.x;
      const long long row = tile * kRows + r;
      const bool live = row < n_rows;
      uint8_t* es = smem + L.e + (it % NE) * ETILE;           // this tile's edge state, updated in place
      // ---- epilogue 0: relu(fmaf(acc0, s_x s_w, b0)) -> int8 codes -> layer-1 operand (R21)
      mbar_wait(&acc0_full[g], j & 1);
      tc_fence_after();
      // etx_dbg_tap_layer: the int32 accumulators of this very kernel, as the tests compare them with the oracle's
      int32_t* tap0 = (a.tap && a.tap_layer == a.l0.index && live) ? a.tap + (size_t)row * D : nullptr;
      int32_t* tap1 = (a.tap && a.tap_layer == a.l1.index && live) ? a.tap + (size_t)row * D : nullptr;
#pragma unroll
      for (int c0 = 0; c0 < D; c0 += 32) {
        uint32_t v[32];
        tmem_ld32(tmem + lane_base + g * D + c0, v);
        store_hidden32<kInt8, KB>(v, c0, scale0, bias0, inv_sx1, Hg, r, tap0);
      }
      tc_fence_before();
      fence_proxy_async();
      mbar_arrive(&hid_full[g]);
      // ---- epilogue 1: fmaf(acc1, s_x s_w, b1) + old e -> e (fp32, in the slot), optional classifier (R14, R16, R21)
      mbar_wait(&acc1_full[g], j & 1);
      tc_fence_after();
      float hacc = 0.0f;
      uint32_t hq_w[4] = {0u, 0u, 0u, 0u};
#pragma unroll
      for (int c0 = 0; c0 < D; c0 += 32) {
        uint32_t v[32];
        tmem_ld32(tmem + lane_base + 2 * D + g * D + c0, v);
        if (tap1) {
#pragma unroll
          for (int jj = 0; jj < 32; ++jj) tap1[c0 + jj] = (int)v[jj];
        }
        if (SB) {
#pragma unroll
          for (int ch = 0; ch < 4; ++ch) {                    // 8 columns = one 16-byte chunk of the bf16 row
            const int c = c0 + ch * 8;
            uint4* p = reinterpret_cast<uint4*>(es + swz<SROW>(r, c / 8));
            const uint4 o = *p;
            float y[8];
#pragma unroll
            for (int jj = 0; jj < 8; ++jj) y[jj] = __fmaf_rn((float)(int)v[ch * 8 + jj], scale1[c + jj], bias1[c + jj]);
            uint4 qv;                                         // fp32 residual add on the widened old state, RNE on store (R14, R21)
            qv.x = pack_bf16x2(__fadd_rn(bf16_lo(o.x), y[0]), __fadd_rn(bf16_hi(o.x), y[1]));
            qv.y = pack_bf16x2(__fadd_rn(bf16_lo(o.y), y[2]), __fadd_rn(bf16_hi(o.y), y[3]));
            qv.z = pack_bf16x2(__fadd_rn(bf16_lo(o.z), y[4]), __fadd_rn(bf16_hi(o.z), y[5]));
            qv.w = pack_bf16x2(__fadd_rn(bf16_lo(o.w), y[6]), __fadd_rn(bf16_hi(o.w), y[7]));
            *p = qv;
            if (NODE && a.hq_out && live) {                   // codes of the stored h for the edge network that follows
              const float is = a.hq_inv_sx;
              hq_w[(ch & 1) * 2 + 0] = pack_i8x4(quant_i8(bf16_lo(qv.x), is), quant_i8(bf16_hi(qv.x), is), quant_i8(bf16_lo(qv.y), is), quant_i8(bf16_hi(qv.y), is));
              hq_w[(ch & 1) * 2 + 1] = pack_i8x4(quant_i8(bf16_lo(qv.z), is), quant_i8(bf16_hi(qv.z), is), quant_i8(bf16_lo(qv.w), is), quant_i8(bf16_hi(qv.w), is));
              if (ch & 1) *reinterpret_cast<uint4*>(a.hq_out + (size_t)row * D + c - 8) = make_uint4(hq_w[0], hq_w[1], hq_w[2], hq_w[3]);
            }
            if (!NODE && a.do_head) {                         // the classifier sees the stored (rounded) state, ascending j (R16)
              hacc = __fmaf_rn(bf16_lo(qv.x), headw[c + 0], hacc); hacc = __fmaf_rn(bf16_hi(qv.x), headw[c + 1], hacc);
              hacc = __fmaf_rn(bf16_lo(qv.y), headw[c + 2], hacc); hacc = __fmaf_rn(bf16_hi(qv.y), headw[c + 3], hacc);
              hacc = __fmaf_rn(bf16_lo(qv.z), headw[c + 4], hacc); hacc = __fmaf_rn(bf16_hi(qv.z), headw[c + 5], hacc);
              hacc = __fmaf_rn(bf16_lo(qv.w), headw[c + 6], hacc); hacc = __fmaf_rn(bf16_hi(qv.w), headw[c + 7], hacc);
            }
          }
        } else
#pragma unroll
        for (int ch = 0; ch < 8; ++ch) {
          const int c = c0 + ch * 4;
          float4* p = reinterpret_cast<float4*>(es + e_off(r, c / 4));
          const float4 o = *p;
          float4 y;
          y.x = __fadd_rn(o.x, __fmaf_rn((float)(int)v[ch * 4 + 0], scale1[c + 0], bias1[c + 0]));
          y.y = __fadd_rn(o.y, __fmaf_rn((float)(int)v[ch * 4 + 1], scale1[c + 1], bias1[c + 1]));
          y.z = __fadd_rn(o.z, __fmaf_rn((float)(int)v[ch * 4 + 2], scale1[c + 2], bias1[c + 2]));
          y.w = __fadd_rn(o.w, __fmaf_rn((float)(int)v[ch * 4 + 3], scale1[c + 3], bias1[c + 3]));
          *p = y;
          if (NODE && a.hq_out && live) {
            const float is = a.hq_inv_sx;
            hq_w[ch & 3] = pack_i8x4(quant_i8(y.x, is), quant_i8(y.y, is), quant_i8(y.z, is), quant_i8(y.w, is));
            if ((ch & 3) == 3) *reinterpret_cast<uint4*>(a.hq_out + (size_t)row * D + c - 12) = make_uint4(hq_w[0], hq_w[1], hq_w[2], hq_w[3]);
          }
          if (!NODE && a.do_head) {                           // ascending j (R16)
            hacc = __fmaf_rn(y.x, headw[c + 0], hacc); hacc = __fmaf_rn(y.y, headw[c + 1], hacc);
            hacc = __fmaf_rn(y.z, headw[c + 2], hacc); hacc = __fmaf_rn(y.w, headw[c + 3], hacc);
          }
        }
      }
      tc_fence_before();                                      // acc1[g] may be overwritten after our next hid_full arrive
      fence_proxy_async();                                    // generic-proxy writes -> visible to the TMA store
      mbar_arrive(&out_ready[it % NE]);
      if (!NODE && a.do_head && live) {
        const float z = __fadd_rn(hacc, head_b);
        a.logit[row] = z;
        a.score[row] = 1.0f / (1.0f + expf(-z));
      }
    }
  }
  tc_fence_before();
  __syncthreads();
  if (warp == kI8MmaWarp) tmem_dealloc(tmem, TMEM_COLS);
}

typedef CUresult (*EncodeTiledFn)(CUtensorMap*, CUtensorMapDataType, cuuint32_t, void*, const cuuint64_t*, const cuuint64_t*,
                                  const cuuint32_t*, const cuuint32_t*, CUtensorMapInterleave, CUtensorMapSwizzle,
                                  CUtensorMapL2promotion, CUtensorMapFloatOOBfill);

template <int D, bool NODE, bool SB>
void edge_i8_launch(etx_ctx* c, const GnnArgs& a, int max_rows, cudaStream_t s) {
  auto kern = edge_net_i8_kernel<D, NODE, SB>;
  constexpr int smem = i8_layout<D, SB>().total + 1024;
  opt_in_smem(c, kern, smem);
  const int tiles = (max_rows + kRows - 1) / kRows;
  const int grid = tiles < c->sm_count ? tiles : c->sm_count;     // one persistent CTA per SM
  if (grid <= 0) return;
  CUtensorMap map;
  memcpy(&map, NODE ? c->h_map : c->e_map, sizeof(map));
  kern<<<grid, kI8Threads, smem, s>>>(map, a);
  c->launches++;
}

}  // namespace

// INT8 mode: tensor map of the fp32 edge state (boxes of 128 rows x 32 floats, 128B swizzle)
bool edge_i8_configure(etx_ctx* c) {
  c->hq = static_cast<int8_t*>(etx_device_alloc(c, (size_t)(c->hp.max_hits > 0 ? c->hp.max_hits : 1) * c->hp.gnn_latent + 256));
  if (!c->hq) return false;
  static_assert(sizeof(CUtensorMap) == sizeof(c->e_map), "etx_ctx::e_map must hold a CUtensorMap");
  void* fn = nullptr;
  cudaDriverEntryPointQueryResult qres;
  if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &fn, cudaEnableDefault, &qres) != cudaSuccess || !fn) return false;
  const int D = c->hp.gnn_latent;
  const bool sb = c->state_bf16;
  const cuuint64_t gstride[1] = {(cuuint64_t)D * (sb ? 2 : 4)};
  const cuuint32_t box[2] = {sb ? (cuuint32_t)D : 32u, (cuuint32_t)kRows};   // fp32: boxes of 32 floats; bf16: the whole row
  const cuuint32_t estr[2] = {1, 1};
  for (int node = 0; node < 2; ++node) {
    const long long rows = node ? c->hp.max_hits : c->max_edges;
    const cuuint64_t gdim[2] = {(cuuint64_t)D, rows > 0 ? (cuuint64_t)rows : 1};
    CUtensorMap map;
    const CUresult r = reinterpret_cast<EncodeTiledFn>(fn)(
        &map, sb ? CU_TENSOR_MAP_DATA_TYPE_BFLOAT16 : CU_TENSOR_MAP_DATA_TYPE_FLOAT32, 2, node ? c->h : c->e, gdim, gstride, box, estr,
        CU_TENSOR_MAP_INTERLEAVE_NONE, (sb && D == 32) ? CU_TENSOR_MAP_SWIZZLE_64B : CU_TENSOR_MAP_SWIZZLE_128B,
        CU_TENSOR_MAP_L2_PROMOTION_L2_256B, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
    if (r != CUDA_SUCCESS) return false;
    memcpy(node ? c->h_map : c->e_map, &map, sizeof(map));
  }
  return true;
}

// INT8 mode (AUTO engine): S4e; the accumulator tap of etx_dbg_tap_layer is served by this kernel itself
void launch_edge_net_i8(etx_ctx* c, int iter, int n_hits, bool do_head, cudaStream_t s) {
  GnnArgs a;
  fill_gnn_args(c, kEdgeNet, iter, n_hits, do_head, a);
  if (do_head && !c->keep_final_state) a.do_head = 2;        // e^L feeds only the classifier: do not write it back
  a.hq_in = c->hq;                                           // written by this iteration's node network (launch_node_net_i8)
  const long long max_rows_ll = (long long)n_hits * c->hp.k;
  const int max_rows = (int)(max_rows_ll > 0x7fffffff ? 0x7fffffff : max_rows_ll);
  if (c->state_bf16) { if (c->hp.gnn_latent == 32) edge_i8_launch<32, false, true>(c, a, max_rows, s); else edge_i8_launch<64, false, true>(c, a, max_rows, s); }
  else { if (c->hp.gnn_latent == 32) edge_i8_launch<32, false, false>(c, a, max_rows, s); else edge_i8_launch<64, false, false>(c, a, max_rows, s); }
}

// S4d in INT8 mode: the same kernel over hits (self state h, second and third segment m_out, m_in)
void launch_node_net_i8(etx_ctx* c, int iter, int n_hits, cudaStream_t s) {
  GnnArgs a;
  fill_gnn_args(c, kNodeNet, iter, n_hits, false, a);
  a.hq_out = c->hq;                                          // codes of the new h under the input scale of this iteration's edge network
  a.hq_inv_sx = c->layers[c->i_iter0 + 4 * iter + 2].dev.inv_sx;
  if (c->state_bf16) { if (c->hp.gnn_latent == 32) edge_i8_launch<32, true, true>(c, a, n_hits, s); else edge_i8_launch<64, true, true>(c, a, n_hits, s); }
  else { if (c->hp.gnn_latent == 32) edge_i8_launch<32, true, false>(c, a, n_hits, s); else edge_i8_launch<64, true, false>(c, a, n_hits, s); }
}

}  // namespace etx
