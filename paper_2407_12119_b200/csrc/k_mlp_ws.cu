// Warp-specialised, software-pipelined tcgen05 kernels for the interaction network's MLPs (S4, bf16 mode).
//
// h0 = MLP(f), e0 = MLP(.), then per step h <- h + MLP([h, m_out, m_in]) and
// e <- e + MLP([h_src, h_dst, e]); the d->1 edge classifier (L80, L142) is fused into the last edge-network
// launch.  The arithmetic and rounding points are exactly those of k_mlp_umma.cu (R3, R14, R16, R20);
// what changes is the schedule.  One persistent CTA per SM, 13 warps in three roles:
//
//   producers  (4 warps)  gather the rows of the next tiles straight into the swizzled UMMA A-tile layout with
//                         16-byte cp.async (h[src] | h[dst] | e, or h | m_out | m_in), kStages tiles deep, so
//                         ~100 KB of loads are in flight per SM at all times (the stage is HBM-bound);
//   MMA issuer (1 thread) tcgen05.mma for layer 0 of tile i+1 is issued before layer 1 of tile i, so the tensor
//                         pipe never waits for an epilogue; accumulators are double-buffered in TMEM;
//   epilogue   (2 x 4 warps) warpgroup g owns tiles i = g (mod 2): TMEM -> registers (tcgen05.ld, lane = row),
//                         bias + ReLU + bf16 -> A tile of layer 1 in shared memory; then bias + residual +
//                         bf16 -> staging -> coalesced 16-byte stores, and the classifier dot product.
//
// mbarriers: full[s] (producers -> MMA), empty[s] (epilogue -> producers: the residual rows have been read and
// layer 0 has finished with the stage), acc0_full[g] / acc1_full[g] (tcgen05.commit -> epilogue),
// h_full[g] (epilogue -> MMA: the layer-1 operand is in shared memory and acc0[g] has been drained).
#include "umma_common.cuh"

namespace etx {

namespace {

using namespace umma;

constexpr int kStages = 3;                  // A-tile ring (48 KB per stage at d = 64)
constexpr int kFeatStages = 8;              // ring of 2 KB feature tiles when layer 0 is the K = 3 FFMA layer
constexpr int kEpiWarps = 8, kProdWarps = 4;
constexpr int kMmaWarp = kEpiWarps + kProdWarps;
constexpr int kWsThreads = (kMmaWarp + 1) * 32;   // 416
// ptxas budgets 65536 / 512 = 128 registers per thread for a 416-thread CTA; the producer warpgroup gives 64 of
// them back (setmaxnreg) and the two epilogue warpgroups take 32 each: 256 * 160 + 128 * 64 + 32 * 128 = 53248.
constexpr int kProdRegs = 64, kEpiRegs = 160;

__device__ __forceinline__ void cp_async16(uint32_t dst, const void* src) {
  asm volatile("cp.async.cg.shared.global [%0], [%1], 16;" ::"r"(dst), "l"(src) : "memory");
}
__device__ __forceinline__ void cp_async_commit() { asm volatile("cp.async.commit_group;" ::: "memory"); }
template <int N>
__device__ __forceinline__ void cp_async_wait() { asm volatile("cp.async.wait_group %0;" ::"n"(N) : "memory"); }

struct WsSmem { int a, h, w0, w1, par, bar, total; };
template <int D>
__host__ __device__ constexpr WsSmem ws_layout() {
  constexpr int SEGB = D * 2;
  WsSmem s{};
  s.a = 0;                                        // kStages x 3 K-blocks [128][SEGB]  (or kFeatStages x [128] float4)
  s.h = s.a + kStages * 3 * kRows * SEGB;         // 2 x [128][SEGB]: layer-1 operand / output staging per warpgroup
  s.w0 = s.h + 2 * kRows * SEGB;                  // W0 image: 3 K-blocks [D][SEGB]
  s.w1 = s.w0 + 3 * D * SEGB;                     // W1 image
  s.par = s.w1 + D * SEGB;                        // fp32: bias0, bias1, head w, W0 of a K = 3 layer (3 x D)
  s.bar = s.par + 6 * D * 4;
  s.total = s.bar + 256;
  return s;
}

// KIND: which network (MlpKind).  L0T: layer 0 is a tensor layer (K = nseg * D gathered segments); otherwise it is
// the K = 3 input layer of an encoder and runs on the FFMA pipe inside the epilogue warps (R20).
template <int KIND, bool L0T, int D>
__global__ void __launch_bounds__(kWsThreads, 1) gnn_mlp_ws_kernel(GnnArgs a) {
  constexpr int KB = D * 2;                                  // bytes per gathered segment row = swizzle width
  constexpr int CPR = KB / 16;                               // 16-byte chunks per segment row
  constexpr int BLK = kRows * KB;                            // one K-block
  constexpr int STAGE = 3 * BLK;
  constexpr WsSmem L = ws_layout<D>();
  constexpr uint32_t TMEM_COLS = 4 * D;                      // acc0[2] | acc1[2]  (128 or 256 columns)
  constexpr bool is_edge = (KIND == kEdgeEnc || KIND == kEdgeNet);
  constexpr bool residual = (KIND == kNodeNet || KIND == kEdgeNet);
  extern __shared__ uint8_t smem_raw[];
  uint8_t* smem = reinterpret_cast<uint8_t*>((reinterpret_cast<uintptr_t>(smem_raw) + 1023) & ~(uintptr_t)1023);
  float* par = reinterpret_cast<float*>(smem + L.par);
  float *bias0 = par, *bias1 = par + D, *headw = par + 2 * D, *w3 = par + 3 * D;
  uint64_t* bars = reinterpret_cast<uint64_t*>(smem + L.bar);
  uint64_t *full = bars, *empty = bars + kFeatStages, *acc0_full = bars + 2 * kFeatStages, *h_full = acc0_full + 2,
           *acc1_full = acc0_full + 4, *bar_w = acc0_full + 6;
  uint32_t* tmem_slot = reinterpret_cast<uint32_t*>(acc0_full + 7);

  const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
  const int nseg = L0T ? a.l0.K / D : 0;                     // 3 (networks) or 2 (the paper's edge encoder, R10)
  const int n_rows = a.n_rows_ptr ? *a.n_rows_ptr : a.n_rows;
  const int n_tiles = (n_rows + kRows - 1) / kRows;
  constexpr int NST = L0T ? kStages : kFeatStages;

  if (tid == 0) {
    for (int s = 0; s < NST; ++s) { mbar_init(&full[s], L0T ? kProdWarps * 32 : 32); mbar_init(&empty[s], 4); }
    for (int g = 0; g < 2; ++g) { mbar_init(&acc0_full[g], 1); mbar_init(&h_full[g], 128); mbar_init(&acc1_full[g], 1); }
    mbar_init(bar_w, 1);
    fence_barrier_init();
  }
  if (warp == kMmaWarp) tmem_alloc(tmem_slot, TMEM_COLS);
  for (int i = tid; i < D; i += kWsThreads) {
    bias0[i] = a.l0.bias[i]; bias1[i] = a.l1.bias[i]; headw[i] = a.head.Wt[i];
    if (!L0T) { w3[i] = a.l0.Wt[i]; w3[D + i] = a.l0.Wt[D + i]; w3[2 * D + i] = a.l0.Wt[2 * D + i]; }
  }
  tc_fence_before();
  __syncthreads();
  tc_fence_after();
  const uint32_t tmem = *tmem_slot;

  if (warp >= kEpiWarps && warp < kMmaWarp) {
    // ================================================================================================ producers
    asm volatile("setmaxnreg.dec.sync.aligned.u32 %0;" ::"n"(kProdRegs));
    const int pw = warp - kEpiWarps;
    if (L0T) {
      constexpr int LAG = kStages - 1;
      int it = 0;
      for (int tile = blockIdx.x; tile < n_tiles; tile += gridDim.x, ++it) {
        const int s = it % kStages;
        const int row = tile * kRows + pw * 32 + lane;
        int is = 0, id = 0;
        if (is_edge && row < n_rows) { is = __ldg(a.src + row); id = __ldg(a.dst + row); }
        mbar_wait(&empty[s], ((it / kStages) & 1) ^ 1);
        const uint32_t st = smem_u32(smem + L.a + s * STAGE);
#pragma unroll
        for (int i = 0; i < CPR; ++i) {
          const int c = i * 32 + lane, rl = c / CPR, piece = c % CPR;
          const int r = pw * 32 + rl;                         // row of the tile
          int grow = tile * kRows + r;
          if (grow >= n_rows) grow = n_rows - 1;              // dead rows of the last tile: any valid row (never stored)
          const int js = __shfl_sync(0xffffffffu, is, rl), jd = __shfl_sync(0xffffffffu, id, rl);
          const uint32_t off = swz<KB>(r, piece);
          const __nv_bfloat16 *p0, *p1, *p2;
          if (KIND == kNodeNet) {
            p0 = static_cast<const __nv_bfloat16*>(a.h) + (size_t)grow * D;
            p1 = static_cast<const __nv_bfloat16*>(a.m) + (size_t)grow * 2 * D;
            p2 = p1 + D;
          } else {
            p0 = static_cast<const __nv_bfloat16*>(a.h) + (size_t)js * D;
            p1 = static_cast<const __nv_bfloat16*>(a.h) + (size_t)jd * D;
            p2 = static_cast<const __nv_bfloat16*>(a.e) + (size_t)grow * D;
          }
          cp_async16(st + off, p0 + piece * 8);
          cp_async16(st + BLK + off, p1 + piece * 8);
          if (nseg > 2) cp_async16(st + 2 * BLK + off, p2 + piece * 8);
        }
        cp_async_commit();
        if (it >= LAG) {                                      // the tile issued LAG iterations ago has landed
          cp_async_wait<LAG>();
          fence_proxy_async();                                // generic-proxy writes -> visible to the tensor core
          mbar_arrive(&full[(it - LAG) % kStages]);
        }
      }
      cp_async_wait<0>();
      fence_proxy_async();
      for (int j = it - (it < LAG ? it : LAG); j < it; ++j) mbar_arrive(&full[j % kStages]);
    } else {
      // K = 3 encoders: producer warp pw stages the features of tiles it = pw (mod 4), 4 rows per lane
      float4* FT = reinterpret_cast<float4*>(smem + L.a);
      for (int it = pw; blockIdx.x + (long long)it * gridDim.x < n_tiles; it += kProdWarps) {
        const int tile = blockIdx.x + it * gridDim.x;
        const int s = it % kFeatStages;
        float4 f[4];
#pragma unroll
        for (int j = 0; j < 4; ++j) {
          const int row = tile * kRows + j * 32 + lane;
          f[j] = make_float4(0.f, 0.f, 0.f, 0.f);
          if (row < n_rows) {
            if (KIND == kNodeEnc) f[j] = __ldg(a.feat + row);
            else {
              const float4 fs = __ldg(a.feat + __ldg(a.src + row)), fd = __ldg(a.feat + __ldg(a.dst + row));
              f[j] = make_float4(fabsf(__fsub_rn(fd.x, fs.x)), fabsf(__fsub_rn(fd.y, fs.y)), fabsf(__fsub_rn(fd.z, fs.z)), 0.f);   // R11
            }
          }
        }
        mbar_wait(&empty[s], ((it / kFeatStages) & 1) ^ 1);
#pragma unroll
        for (int j = 0; j < 4; ++j) FT[s * kRows + j * 32 + lane] = f[j];
        mbar_arrive(&full[s]);
      }
    }
  } else if (warp == kMmaWarp) {
    // ================================================================================================ MMA issuer
    if (elect_one()) {
      const uint32_t b0 = L0T ? (uint32_t)(nseg * D * KB) : 0u, b1 = (uint32_t)(D * KB);
      mbar_expect_tx(bar_w, b0 + b1);
      if (L0T) bulk_g2s(smem + L.w0, a.l0.Wtc, b0, bar_w);
      bulk_g2s(smem + L.w1, a.l1.Wtc, b1, bar_w);
      mbar_wait(bar_w, 0);
      const uint32_t idesc = make_idesc<kBf16>(D);
      const uint32_t a_addr = smem_u32(smem + L.a), h_addr = smem_u32(smem + L.h);
      const uint32_t w0_addr = smem_u32(smem + L.w0), w1_addr = smem_u32(smem + L.w1);
      auto layer1 = [&](int j) {                              // layer 1 of the CTA's j-th tile
        const int g = j & 1;
        mbar_wait(&h_full[g], (j >> 1) & 1);
        tc_fence_after();
        issue_layer<kBf16, KB>(h_addr + g * BLK, w1_addr, KB, D, tmem + 2 * D + g * D, idesc);
        umma_commit(&acc1_full[g]);
      };
      int it = 0;
      for (int tile = blockIdx.x; tile < n_tiles; tile += gridDim.x, ++it) {
        if (L0T) {
          const int s = it % kStages, g = it & 1;
          mbar_wait(&full[s], (it / kStages) & 1);
          tc_fence_after();
          // acc0[g] was drained by epilogue 0 of tile it-2, which h_full (waited on for layer 1 of it-2) covers
          issue_layer<kBf16, KB>(a_addr + s * STAGE, w0_addr, nseg * KB, D, tmem + g * D, idesc);
          umma_commit(&acc0_full[g]);
          if (it > 0) layer1(it - 1);
        } else {
          layer1(it);
        }
      }
      if (L0T && it > 0) layer1(it - 1);
    }
  } else {
    // ================================================================================================ epilogue
    asm volatile("setmaxnreg.inc.sync.aligned.u32 %0;" ::"n"(kEpiRegs));
    const int g = warp >> 2, q = warp & 3;                    // warpgroup, TMEM lane quarter
    const int r = q * 32 + lane;                              // row of the tile owned by this thread
    const uint32_t lane_base = (uint32_t)(q * 32) << 16;
    uint8_t* Hg = smem + L.h + g * BLK;
    const float head_b = a.head.bias[0];
    __nv_bfloat16* state = static_cast<__nv_bfloat16*>(is_edge ? a.e : a.h);
    int j = 0;                                                // this warpgroup's tile counter
    for (int it = g; blockIdx.x + (long long)it * gridDim.x < n_tiles; it += 2, ++j) {
      const int tile = blockIdx.x + it * gridDim.x;
      const int row = tile * kRows + r;
      const bool live = row < n_rows;
      uint4 res[CPR];                                         // this row's old state (residual operand), bf16
      if (L0T) {
        const int s = it % kStages;
        mbar_wait(&acc0_full[g], j & 1);
        tc_fence_after();
        if (residual) {
          const uint8_t* seg = smem + L.a + s * STAGE + (KIND == kNodeNet ? 0 : 2) * BLK;
#pragma unroll
          for (int c = 0; c < CPR; ++c) res[c] = *reinterpret_cast<const uint4*>(seg + swz<KB>(r, c));
        }
        __syncwarp();
        if (lane == 0) mbar_arrive(&empty[s]);                // layer 0 is done with the stage and so are we
        // ---- epilogue 0: relu(acc0 + b0) -> bf16 -> layer-1 operand (R3, R20)
#pragma unroll
        for (int c0 = 0; c0 < D; c0 += 32) {
          uint32_t v[32];
          tmem_ld32(tmem + lane_base + g * D + c0, v);
          float y[32];
#pragma unroll
          for (int jj = 0; jj < 32; jj += 4) {
            const float4 b = *reinterpret_cast<const float4*>(bias0 + c0 + jj);
            y[jj + 0] = fmaxf(__fadd_rn(__uint_as_float(v[jj + 0]), b.x), 0.0f);
            y[jj + 1] = fmaxf(__fadd_rn(__uint_as_float(v[jj + 1]), b.y), 0.0f);
            y[jj + 2] = fmaxf(__fadd_rn(__uint_as_float(v[jj + 2]), b.z), 0.0f);
            y[jj + 3] = fmaxf(__fadd_rn(__uint_as_float(v[jj + 3]), b.w), 0.0f);
          }
          store_operand32<kBf16, KB>(y, c0, 0.0f, Hg, r);
        }
      } else {
        // ---- K = 3 input layer on the FFMA pipe, pinned order (R3, R20)
        const int s = it % kFeatStages;
        mbar_wait(&full[s], (it / kFeatStages) & 1);
        const float4 f = reinterpret_cast<const float4*>(smem + L.a)[s * kRows + r];
        __syncwarp();
        if (lane == 0) mbar_arrive(&empty[s]);
#pragma unroll
        for (int c0 = 0; c0 < D; c0 += 32) {
          float y[32];
#pragma unroll
          for (int jj = 0; jj < 32; ++jj) {
            float acc = __fmaf_rn(f.x, w3[c0 + jj], 0.0f);
            acc = __fmaf_rn(f.y, w3[D + c0 + jj], acc);
            acc = __fmaf_rn(f.z, w3[2 * D + c0 + jj], acc);
            y[jj] = fmaxf(__fadd_rn(acc, bias0[c0 + jj]), 0.0f);
          }
          store_operand32<kBf16, KB>(y, c0, 0.0f, Hg, r);
        }
      }
      tc_fence_before();
      fence_proxy_async();
      mbar_arrive(&h_full[g]);
      // ---- epilogue 1: acc1 + b1 (+ old state), bf16 store, optional classifier (R14, R16, R20)
      mbar_wait(&acc1_full[g], j & 1);
      tc_fence_after();
      float hacc = 0.0f;
#pragma unroll
      for (int c0 = 0; c0 < D; c0 += 32) {
        uint32_t v[32];
        tmem_ld32(tmem + lane_base + 2 * D + g * D + c0, v);
#pragma unroll
        for (int ch = 0; ch < 4; ++ch) {
          float y[8];
          const float4 ba = *reinterpret_cast<const float4*>(bias1 + c0 + ch * 8), bb = *reinterpret_cast<const float4*>(bias1 + c0 + ch * 8 + 4);
          y[0] = __fadd_rn(__uint_as_float(v[ch * 8 + 0]), ba.x); y[1] = __fadd_rn(__uint_as_float(v[ch * 8 + 1]), ba.y);
          y[2] = __fadd_rn(__uint_as_float(v[ch * 8 + 2]), ba.z); y[3] = __fadd_rn(__uint_as_float(v[ch * 8 + 3]), ba.w);
          y[4] = __fadd_rn(__uint_as_float(v[ch * 8 + 4]), bb.x); y[5] = __fadd_rn(__uint_as_float(v[ch * 8 + 5]), bb.y);
          y[6] = __fadd_rn(__uint_as_float(v[ch * 8 + 6]), bb.z); y[7] = __fadd_rn(__uint_as_float(v[ch * 8 + 7]), bb.w);
          if (residual) {
            const uint4 o = res[c0 / 8 + ch];
            y[0] = __fadd_rn(bf16_lo(o.x), y[0]); y[1] = __fadd_rn(bf16_hi(o.x), y[1]);
            y[2] = __fadd_rn(bf16_lo(o.y), y[2]); y[3] = __fadd_rn(bf16_hi(o.y), y[3]);
            y[4] = __fadd_rn(bf16_lo(o.z), y[4]); y[5] = __fadd_rn(bf16_hi(o.z), y[5]);
            y[6] = __fadd_rn(bf16_lo(o.w), y[6]); y[7] = __fadd_rn(bf16_hi(o.w), y[7]);
          }
          uint4 qv;
          qv.x = pack_bf16x2(y[0], y[1]); qv.y = pack_bf16x2(y[2], y[3]);
          qv.z = pack_bf16x2(y[4], y[5]); qv.w = pack_bf16x2(y[6], y[7]);
          *reinterpret_cast<uint4*>(Hg + swz<KB>(r, c0 / 8 + ch)) = qv;        // staging (layer 1 has finished with Hg)
          if (is_edge && a.do_head) {                         // the classifier sees the stored bf16 state (R20), ascending j (R16)
            const float* hw = headw + c0 + ch * 8;
            hacc = __fmaf_rn(bf16_lo(qv.x), hw[0], hacc); hacc = __fmaf_rn(bf16_hi(qv.x), hw[1], hacc);
            hacc = __fmaf_rn(bf16_lo(qv.y), hw[2], hacc); hacc = __fmaf_rn(bf16_hi(qv.y), hw[3], hacc);
            hacc = __fmaf_rn(bf16_lo(qv.z), hw[4], hacc); hacc = __fmaf_rn(bf16_hi(qv.z), hw[5], hacc);
            hacc = __fmaf_rn(bf16_lo(qv.w), hw[6], hacc); hacc = __fmaf_rn(bf16_hi(qv.w), hw[7], hacc);
          }
        }
      }
      tc_fence_before();                                      // acc1[g] may be overwritten after our next h_full arrive
      __syncwarp();
      // ---- coalesced copy-out of this warp's 32 rows: each instruction stores 32 x 16 B = 32 / CPR full rows
#pragma unroll
      for (int i = 0; i < CPR; ++i) {
        const int c = i * 32 + lane, rl = c / CPR, piece = c % CPR;
        const int rr = q * 32 + rl;
        const long long grow = (long long)tile * kRows + rr;
        if (grow < n_rows)
          *reinterpret_cast<uint4*>(state + (size_t)grow * D + piece * 8) = *reinterpret_cast<const uint4*>(Hg + swz<KB>(rr, piece));
      }
      if (is_edge && a.do_head && live) {
        const float z = __fadd_rn(hacc, head_b);
        a.logit[row] = z;
        a.score[row] = 1.0f / (1.0f + expf(-z));
      }
      __syncwarp();                                           // staging rows are warp-private: safe to overwrite next tile
    }
  }
  tc_fence_before();
  __syncthreads();
  if (warp == kMmaWarp) tmem_dealloc(tmem, TMEM_COLS);
}

template <int KIND, bool L0T, int D>
void ws_launch_one(etx_ctx* c, const GnnArgs& a, int max_rows, cudaStream_t s) {
  auto kern = gnn_mlp_ws_kernel<KIND, L0T, D>;
  constexpr int smem = ws_layout<D>().total + 1024;
  opt_in_smem(c, kern, smem);
  const int tiles = (max_rows + kRows - 1) / kRows;
  const int grid = tiles < c->sm_count ? tiles : c->sm_count;     // one persistent CTA per SM
  if (grid <= 0) return;
  kern<<<grid, kWsThreads, smem, s>>>(a);
  c->launches++;
}

template <int D>
void ws_launch_kind(etx_ctx* c, int kind, const GnnArgs& a, int max_rows, cudaStream_t s) {
  const bool l0t = a.l0.tensor != 0;
  switch (kind) {
    case kNodeEnc: ws_launch_one<kNodeEnc, false, D>(c, a, max_rows, s); break;
    case kEdgeEnc:
      if (l0t) ws_launch_one<kEdgeEnc, true, D>(c, a, max_rows, s);
      else ws_launch_one<kEdgeEnc, false, D>(c, a, max_rows, s);
      break;
    case kNodeNet: ws_launch_one<kNodeNet, true, D>(c, a, max_rows, s); break;
    default:       ws_launch_one<kEdgeNet, true, D>(c, a, max_rows, s); break;
  }
}

}  // namespace

// bf16 mode only (state rows are bf16, so the gather is a plain 16-byte copy).
void launch_gnn_mlp_ws(etx_ctx* c, int kind, int iter, int n_hits, bool do_head, cudaStream_t s) {
  GnnArgs a;
  fill_gnn_args(c, kind, iter, n_hits, do_head, a);
  const bool is_edge = (kind == kEdgeEnc || kind == kEdgeNet);
  const long long max_rows_ll = is_edge ? (long long)n_hits * c->hp.k : n_hits;
  const int max_rows = (int)(max_rows_ll > 0x7fffffff ? 0x7fffffff : max_rows_ll);
  if (c->hp.gnn_latent == 32) ws_launch_kind<32>(c, kind, a, max_rows, s);
  else ws_launch_kind<64>(c, kind, a, max_rows, s);
}

}  // namespace etx
