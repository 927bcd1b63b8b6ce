// S4e, INT8 mode (R21): e <- e + MLP_k([h_src, h_dst, e]) with int8 operands, int32 accumulation on
// tcgen05 (kind::i8), fp32 dequantisation + bias + ReLU, fp32 state.  PAPER.md L140, L148; the paper quantised only
// its embedding (L265-269) and names the GNN as the step where INT8 would pay most (L271).
//
// Same arithmetic, operation for operation, as gnn_mlp_umma_kernel<kEdgeNet, kInt8, D> (every int32 accumulator is
// reproduced bit for bit, and every other op is a single pinned fp32 op), but warp-specialised and pipelined:
//
//   producers  (8 warps)  read the fp32 rows h[src] | h[dst] | e of the next tiles, quantise them
//                         (q = clamp(rne(x * (1 / s_x)), +-127)) and write the int8 A tile in the swizzled UMMA
//                         layout, kI8Stages tiles ahead -- the quantisation is ~1,000 ALU instructions per row and
//                         is what the serial kernel could not hide;
//   MMA issuer (1 thread) layer 0 of tile i+1 is issued before layer 1 of tile i; accumulators double-buffered in TMEM;
//   epilogue   (2 x 4 warps) warpgroup g owns tiles i = g (mod 2): acc0 -> fmaf(acc, s_x s_w, b) -> relu -> int8 ->
//                         layer-1 operand; acc1 -> fmaf -> + old e (fp32, re-read: an L2 hit) -> e, and the
//                         classifier dot product on the last step.
#include "umma_common.cuh"

namespace etx {

namespace {

using namespace umma;

constexpr int kI8Stages = 4;
constexpr int kI8EpiWarps = 8, kI8ProdWarps = 8;
constexpr int kI8MmaWarp = kI8EpiWarps + kI8ProdWarps;
constexpr int kI8Threads = (kI8MmaWarp + 1) * 32;          // 544
constexpr int kI8ProdThreads = kI8ProdWarps * 32;
// ptxas compiles the 544-thread CTA with 96 registers per thread; the two producer warpgroups hand 16 each to the
// two epilogue warpgroups: 256 * 80 + 256 * 112 + 32 * 96 = 52224 = 544 * 96.
constexpr int kI8ProdRegs = 80, kI8EpiRegs = 112;

struct I8Smem { int a, h, stg, w0, w1, par, bar, total; };
template <int D>
__host__ __device__ constexpr I8Smem i8_layout() {
  I8Smem s{};
  s.a = 0;                                   // kI8Stages x 3 K-blocks [128][D] int8
  s.h = s.a + kI8Stages * 3 * kRows * D;     // 2 x [128][D]: layer-1 operand per epilogue warpgroup
  s.stg = s.h + 2 * kRows * D;               // 2 x [128][D] fp32: output staging per epilogue warpgroup (chunk-swizzled)
  s.w0 = s.stg + 2 * kRows * D * 4;          // W0 image: 3 K-blocks [D][D]
  s.w1 = s.w0 + 3 * D * D;                   // W1 image
  s.par = s.w1 + D * D;                      // fp32: scale0, bias0, scale1, bias1, head w
  s.bar = s.par + 5 * D * 4;
  s.total = s.bar + 128;
  return s;
}

template <int D>
__global__ void __launch_bounds__(kI8Threads, 1) edge_net_i8_kernel(GnnArgs a) {
  constexpr int KB = D;                                      // bytes per int8 segment row = swizzle width (32 / 64)
  constexpr int CPR = KB / 16;                               // 16-byte chunks per segment row
  constexpr int BLK = kRows * KB;
  constexpr int STAGE = 3 * BLK;
  constexpr I8Smem L = i8_layout<D>();
  constexpr uint32_t TMEM_COLS = 4 * D;                      // acc0[2] | acc1[2]
  extern __shared__ uint8_t smem_raw[];
  uint8_t* smem = reinterpret_cast<uint8_t*>((reinterpret_cast<uintptr_t>(smem_raw) + 1023) & ~(uintptr_t)1023);
  float* par = reinterpret_cast<float*>(smem + L.par);
  float *scale0 = par, *bias0 = par + D, *scale1 = par + 2 * D, *bias1 = par + 3 * D, *headw = par + 4 * D;
  uint64_t* bars = reinterpret_cast<uint64_t*>(smem + L.bar);
  uint64_t *full = bars, *empty = bars + kI8Stages, *acc0_full = bars + 2 * kI8Stages, *hid_full = acc0_full + 2,
           *acc1_full = acc0_full + 4, *bar_w = acc0_full + 6;
  uint32_t* tmem_slot = reinterpret_cast<uint32_t*>(acc0_full + 7);

  const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
  const int n_rows = *a.n_rows_ptr;
  const int n_tiles = (n_rows + kRows - 1) / kRows;

  if (tid == 0) {
    for (int s = 0; s < kI8Stages; ++s) { mbar_init(&full[s], kI8ProdThreads); mbar_init(&empty[s], 1); }
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

  if (warp >= kI8EpiWarps && warp < kI8MmaWarp) {
    // ================================================================================================ producers
    asm volatile("setmaxnreg.dec.sync.aligned.u32 %0;" ::"n"(kI8ProdRegs));
    const int pt = tid - kI8EpiWarps * 32;                   // 0 .. 255
    const float inv_sx0 = a.l0.inv_sx;
    const float* hbase = static_cast<const float*>(a.h);
    const float* ebase = static_cast<const float*>(a.e);
    int it = 0;
    for (int tile = blockIdx.x; tile < n_tiles; tile += gridDim.x, ++it) {
      const int s = it % kI8Stages;
      mbar_wait(&empty[s], ((it / kI8Stages) & 1) ^ 1);
      uint8_t* st = smem + L.a + s * STAGE;
      // item c = (row r, 16-byte chunk `piece` of the int8 row) = 16 consecutive fp32 of the source row; CPR
      // consecutive threads share a row, so a warp reads 32 / CPR whole rows (coalesced for the contiguous e tile)
#pragma unroll
      for (int i = 0; i < (kRows * CPR) / kI8ProdThreads; ++i) {
        const int c = i * kI8ProdThreads + pt, r = c / CPR, piece = c % CPR;
        int grow = tile * kRows + r;
        if (grow >= n_rows) grow = n_rows - 1;                // dead rows of the last tile: any valid row (never stored)
        const int js = __ldg(a.src + grow), jd = __ldg(a.dst + grow);
        const float* p[3] = {hbase + (size_t)js * D + piece * 16, hbase + (size_t)jd * D + piece * 16,
                             ebase + (size_t)grow * D + piece * 16};
#pragma unroll
        for (int sg = 0; sg < 3; ++sg) {
          const float4* q4 = reinterpret_cast<const float4*>(p[sg]);
          const float4 f0 = __ldg(q4), f1 = __ldg(q4 + 1), f2 = __ldg(q4 + 2), f3 = __ldg(q4 + 3);
          uint4 q;
          q.x = pack_i8x4(quant_i8(f0.x, inv_sx0), quant_i8(f0.y, inv_sx0), quant_i8(f0.z, inv_sx0), quant_i8(f0.w, inv_sx0));
          q.y = pack_i8x4(quant_i8(f1.x, inv_sx0), quant_i8(f1.y, inv_sx0), quant_i8(f1.z, inv_sx0), quant_i8(f1.w, inv_sx0));
          q.z = pack_i8x4(quant_i8(f2.x, inv_sx0), quant_i8(f2.y, inv_sx0), quant_i8(f2.z, inv_sx0), quant_i8(f2.w, inv_sx0));
          q.w = pack_i8x4(quant_i8(f3.x, inv_sx0), quant_i8(f3.y, inv_sx0), quant_i8(f3.z, inv_sx0), quant_i8(f3.w, inv_sx0));
          *reinterpret_cast<uint4*>(st + sg * BLK + swz<KB>(r, piece)) = q;
        }
      }
      fence_proxy_async();                                    // generic-proxy writes -> visible to the tensor core
      mbar_arrive(&full[s]);
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
        const int s = it % kI8Stages, g = it & 1;
        mbar_wait(&full[s], (it / kI8Stages) & 1);
        tc_fence_after();
        // acc0[g] was drained by epilogue 0 of tile it-2, which hid_full (waited on for layer 1 of it-2) covers
        issue_layer<kInt8, KB>(a_addr + s * STAGE, w0_addr, 3 * KB, D, tmem + g * D, idesc);
        umma_commit(&acc0_full[g]);
        umma_commit(&empty[s]);                               // layer 0 is the stage's only reader
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
    uint8_t* Sg = smem + L.stg + g * (kRows * D * 4);         // fp32 staging tile of this warpgroup
    auto stg_off = [](int row_, int chunk) { return row_ * (D * 4) + ((chunk ^ (row_ & (D / 4 - 1))) << 4); };
    const float head_b = a.head.bias[0];
    const float inv_sx1 = a.l1.inv_sx;
    float* state = static_cast<float*>(a.e);
    int j = 0;                                                // this warpgroup's tile counter
    for (int it = g; blockIdx.x + (long long)it * gridDim.x < n_tiles; it += 2, ++j) {
      const long long tile = blockIdx.x + (long long)it * gridDim.x;
      const long long row = tile * kRows + r;
      const bool live = row < n_rows;
      // ---- epilogue 0: relu(fmaf(acc0, s_x s_w, b0)) -> int8 codes -> layer-1 operand (R21)
      mbar_wait(&acc0_full[g], j & 1);
      tc_fence_after();
#pragma unroll
      for (int c0 = 0; c0 < D; c0 += 32) {
        uint32_t v[32];
        tmem_ld32(tmem + lane_base + g * D + c0, v);
        store_hidden32<kInt8, KB>(v, c0, scale0, bias0, inv_sx1, Hg, r, nullptr);
      }
      tc_fence_before();
      fence_proxy_async();
      mbar_arrive(&hid_full[g]);
      // ---- epilogue 1: fmaf(acc1, s_x s_w, b1) + old e -> e (fp32), optional classifier (R14, R16, R21).
      //      The thread that owns a row dequantises it into a shared staging tile; the residual add and the store
      //      then run over the tile in global-memory order (16 bytes per thread, whole rows per group of threads):
      //      a row-per-thread read-modify-write of e cost a third of the kernel.
      mbar_wait(&acc1_full[g], j & 1);
      tc_fence_after();
#pragma unroll
      for (int c0 = 0; c0 < D; c0 += 32) {
        uint32_t v[32];
        tmem_ld32(tmem + lane_base + 2 * D + g * D + c0, v);
#pragma unroll
        for (int ch = 0; ch < 8; ++ch) {
          float4 y;
          const int c = c0 + ch * 4;
          y.x = __fmaf_rn((float)(int)v[ch * 4 + 0], scale1[c + 0], bias1[c + 0]);
          y.y = __fmaf_rn((float)(int)v[ch * 4 + 1], scale1[c + 1], bias1[c + 1]);
          y.z = __fmaf_rn((float)(int)v[ch * 4 + 2], scale1[c + 2], bias1[c + 2]);
          y.w = __fmaf_rn((float)(int)v[ch * 4 + 3], scale1[c + 3], bias1[c + 3]);
          *reinterpret_cast<float4*>(Sg + stg_off(r, c / 4)) = y;
        }
      }
      tc_fence_before();                                      // acc1[g] may be overwritten after our next hid_full arrive
      asm volatile("bar.sync %0, 128;" ::"r"(1 + g) : "memory");
      {
        constexpr int CH = D / 4;                             // 16-byte chunks per row = threads per row
        const int t = (warp & 3) * 32 + lane, cc = t % CH;
#pragma unroll 4
        for (int rr = t / CH; rr < kRows; rr += 128 / CH) {
          const long long grow = tile * kRows + rr;
          if (grow < n_rows) {
            float* gp = state + (size_t)grow * D + cc * 4;
            const float4 o = *reinterpret_cast<const float4*>(gp);
            float4 y = *reinterpret_cast<const float4*>(Sg + stg_off(rr, cc));
            y.x = __fadd_rn(o.x, y.x); y.y = __fadd_rn(o.y, y.y); y.z = __fadd_rn(o.z, y.z); y.w = __fadd_rn(o.w, y.w);
            *reinterpret_cast<float4*>(gp) = y;
            if (a.do_head) *reinterpret_cast<float4*>(Sg + stg_off(rr, cc)) = y;
          }
        }
      }
      if (a.do_head) {                                        // the classifier: ascending j over the row's new state (R16)
        asm volatile("bar.sync %0, 128;" ::"r"(1 + g) : "memory");
        if (live) {
          float hacc = 0.0f;
#pragma unroll
          for (int c4 = 0; c4 < D / 4; ++c4) {
            const float4 y = *reinterpret_cast<const float4*>(Sg + stg_off(r, c4));
            hacc = __fmaf_rn(y.x, headw[c4 * 4 + 0], hacc); hacc = __fmaf_rn(y.y, headw[c4 * 4 + 1], hacc);
            hacc = __fmaf_rn(y.z, headw[c4 * 4 + 2], hacc); hacc = __fmaf_rn(y.w, headw[c4 * 4 + 3], hacc);
          }
          const float z = __fadd_rn(hacc, head_b);
          a.logit[row] = z;
          a.score[row] = 1.0f / (1.0f + expf(-z));
        }
      }
      asm volatile("bar.sync %0, 128;" ::"r"(1 + g) : "memory");   // the staging tile is free for the next tile
    }
  }
  tc_fence_before();
  __syncthreads();
  if (warp == kI8MmaWarp) tmem_dealloc(tmem, TMEM_COLS);
}

template <int D>
void edge_i8_launch(etx_ctx* c, const GnnArgs& a, int max_rows, cudaStream_t s) {
  auto kern = edge_net_i8_kernel<D>;
  constexpr int smem = i8_layout<D>().total + 1024;
  static bool configured = false;
  if (!configured) { cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, smem); configured = true; }
  const int tiles = (max_rows + kRows - 1) / kRows;
  const int grid = tiles < c->sm_count ? tiles : c->sm_count;     // one persistent CTA per SM
  if (grid <= 0) return;
  kern<<<grid, kI8Threads, smem, s>>>(a);
  c->launches++;
}

}  // namespace

// INT8 mode, fp32 state, no accumulator tap requested (the tap stays with gnn_mlp_umma_kernel)
void launch_edge_net_i8(etx_ctx* c, int iter, int n_hits, bool do_head, cudaStream_t s) {
  GnnArgs a;
  fill_gnn_args(c, kEdgeNet, iter, n_hits, do_head, a);
  const long long max_rows_ll = (long long)n_hits * c->hp.k;
  const int max_rows = (int)(max_rows_ll > 0x7fffffff ? 0x7fffffff : max_rows_ll);
  if (c->hp.gnn_latent == 32) edge_i8_launch<32>(c, a, max_rows, s);
  else edge_i8_launch<64>(c, a, max_rows, s);
}

}  // namespace etx
