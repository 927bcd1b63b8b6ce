// S4e, bf16 mode: the interaction network's edge update  e <- e + MLP_k([h_src, h_dst, e])  (PAPER.md L140,
// L148) and, on the last step, the d -> 1 edge classifier (L80, L142), as one persistent tcgen05 kernel whose
// edge-state traffic is moved entirely by TMA.
//
// This is the kernel that decides the step time: per launch it must read and write the whole edge state
// (2 * E * d * 2 bytes, 2.5 GB at cfg 2), so everything is arranged to keep HBM requests in flight and the
// per-tile epilogue short:
//
//   * the tile of `e` being updated (128 consecutive rows = one contiguous 16 KB block) is loaded by one TMA
//     instruction into a 128B-swizzled slot of a 5-deep ring, updated IN PLACE in shared memory by the epilogue,
//     and written back by one TMA store from the same slot;
//   * h[src] and h[dst] (L2-resident: edges are sorted by src and dst lies in the same event) are gathered with
//     16-byte cp.async into a separate 3-deep ring, so the depth of the HBM ring does not pay for them;
//   * bias and residual are folded into the MMAs: acc0 = 1 * b0' + [h_src | h_dst | e] * W0^T and
//     acc1 = 1 * b1' + hidden * W1^T + e * I, where b' is the fp32 bias split exactly into three bf16 terms and I
//     is the identity (a bf16 value times 1.0 is exact in the fp32 accumulator).  The epilogues are then
//     TMEM -> cvt(.relu).bf16x2 -> store and nothing else;
//   * the hidden activations never touch shared memory: epilogue 0 writes them back to tensor memory (two bf16
//     per 32-bit column, tcgen05.st) and layer 1 takes its A operand from there, so the gather slot is released
//     as soon as layer 0 has finished;
//   * every tcgen05.mma / commit is issued under elect.sync, which lets ptxas keep descriptors and tensor-memory
//     addresses in uniform registers (with `lane == 0` each MMA cost an ELECT / R2UR.BROADCAST loop, ~75 cycles,
//     and the issuing thread was the bottleneck: 22 MMAs per tile).
//
// Rounding points are those of DESIGN.md R20 (operands and stored state bf16 RNE, accumulation fp32); the order of
// the fp32 additions inside the tensor core is not specified, which the bf16 tolerance covers.
//
// Warp roles (15 warps, one CTA per SM):
//   0-7   epilogue, two warpgroups; warpgroup g owns the CTA's tiles it = g (mod 2)
//   8-10  gather producers (cp.async), one per slot of the gather ring; warp 11 only donates registers
//   12    MMA issuer (one elected thread)
//   13    TMA loader (one thread)       14    TMA storer (one thread)
// mbarriers: self_full / self_empty / out_ready [kNE] (TMA load -> MMA, TMA store read -> loader, epilogue 1 ->
// storer), aux_full / aux_empty [kNH] (gather -> MMA, tcgen05.commit after layer 0 -> gather), acc0_full /
// hid_full / acc1_full [2] (commit -> epilogue 0, epilogue 0 -> MMA, commit -> epilogue 1).
#include <cuda.h>
#include <string.h>

#include "umma_common.cuh"

namespace etx {

namespace {

using namespace umma;

constexpr int kNE = 5;                      // ring of edge-state tiles (HBM latency)
constexpr int kNH = 3;                      // ring of gathered [h_src | h_dst] tile pairs (L2 latency)
constexpr int kEpiWarps = 8, kGatherWarps = 4;
constexpr int kMmaWarp = kEpiWarps + kGatherWarps, kLoadWarp = kMmaWarp + 1, kStoreWarp = kMmaWarp + 2;
constexpr int kThreads = (kStoreWarp + 1) * 32;   // 480
// ptxas budgets 65536 / 512 = 128 registers per thread; the gather warpgroup hands 64 of them back and the two
// epilogue warpgroups take 32 each: 256 * 160 + 128 * 64 + 96 * 128 = 61440 = 480 * 128.
constexpr int kGatherRegs = 64, kEpiRegs = 160;

__device__ __forceinline__ void cp_async16(uint32_t dst, const void* src) {
  asm volatile("cp.async.cg.shared.global [%0], [%1], 16;" ::"r"(dst), "l"(src) : "memory");
}
__device__ __forceinline__ void cp_async_commit() { asm volatile("cp.async.commit_group;" ::: "memory"); }
template <int N>
__device__ __forceinline__ void cp_async_wait() { asm volatile("cp.async.wait_group %0;" ::"n"(N) : "memory"); }

// TMA: one box of a 2-D tensor (inner coordinate x, row y) global -> shared, completing on an mbarrier
__device__ __forceinline__ void tma_load_2d(uint32_t dst, const CUtensorMap* map, int x, int y, uint64_t* bar) {
  asm volatile("cp.async.bulk.tensor.2d.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1, {%3, %4}], [%2];"
               ::"r"(dst), "l"(reinterpret_cast<uint64_t>(map)), "r"(smem_u32(bar)), "r"(x), "r"(y) : "memory");
}
// TMA: shared -> global, tracked by the issuing thread's bulk async-group
__device__ __forceinline__ void tma_store_2d(const CUtensorMap* map, uint32_t src, int x, int y) {
  asm volatile("cp.async.bulk.tensor.2d.global.shared::cta.bulk_group [%0, {%2, %3}], [%1];"
               ::"l"(reinterpret_cast<uint64_t>(map)), "r"(src), "r"(x), "r"(y) : "memory");
}
__device__ __forceinline__ void bulk_commit() { asm volatile("cp.async.bulk.commit_group;" ::: "memory"); }
__device__ __forceinline__ void bulk_wait_read0() { asm volatile("cp.async.bulk.wait_group.read 0;" ::: "memory"); }
__device__ __forceinline__ void bulk_wait0() { asm volatile("cp.async.bulk.wait_group 0;" ::: "memory"); }

__device__ __forceinline__ void tmem_st32(uint32_t taddr, const uint32_t (&v)[32]) {
  asm volatile(
      "tcgen05.st.sync.aligned.32x32b.x32.b32 [%0], "
      "{%1, %2, %3, %4, %5, %6, %7, %8, %9, %10, %11, %12, %13, %14, %15, %16, "
      "%17, %18, %19, %20, %21, %22, %23, %24, %25, %26, %27, %28, %29, %30, %31, %32};"
      :: "r"(taddr), "r"(v[0]), "r"(v[1]), "r"(v[2]), "r"(v[3]), "r"(v[4]), "r"(v[5]), "r"(v[6]), "r"(v[7]),
         "r"(v[8]), "r"(v[9]), "r"(v[10]), "r"(v[11]), "r"(v[12]), "r"(v[13]), "r"(v[14]), "r"(v[15]),
         "r"(v[16]), "r"(v[17]), "r"(v[18]), "r"(v[19]), "r"(v[20]), "r"(v[21]), "r"(v[22]), "r"(v[23]),
         "r"(v[24]), "r"(v[25]), "r"(v[26]), "r"(v[27]), "r"(v[28]), "r"(v[29]), "r"(v[30]), "r"(v[31]) : "memory");
}
__device__ __forceinline__ void tmem_st16(uint32_t taddr, const uint32_t (&v)[32]) {
  asm volatile(
      "tcgen05.st.sync.aligned.32x32b.x16.b32 [%0], "
      "{%1, %2, %3, %4, %5, %6, %7, %8, %9, %10, %11, %12, %13, %14, %15, %16};"
      :: "r"(taddr), "r"(v[0]), "r"(v[1]), "r"(v[2]), "r"(v[3]), "r"(v[4]), "r"(v[5]), "r"(v[6]), "r"(v[7]),
         "r"(v[8]), "r"(v[9]), "r"(v[10]), "r"(v[11]), "r"(v[12]), "r"(v[13]), "r"(v[14]), "r"(v[15]) : "memory");
}
__device__ __forceinline__ void tmem_st_wait() { asm volatile("tcgen05.wait::st.sync.aligned;" ::: "memory"); }

// D[tmem] (+)= A[tmem] * B[smem]^T: A is a 128-lane x K block of tensor memory, two bf16 per 32-bit column
__device__ __forceinline__ void umma_ts(uint32_t tmem_d, uint32_t tmem_a, uint64_t bdesc, uint32_t idesc, uint32_t accumulate) {
  asm volatile("{\n\t.reg .pred p;\n\tsetp.ne.b32 p, %4, 0;\n\t"
               "tcgen05.mma.cta_group::1.kind::f16 [%0], [%1], %2, %3, p;\n\t}"
               ::"r"(tmem_d), "r"(tmem_a), "l"(bdesc), "r"(idesc), "r"(accumulate) : "memory");
}

struct EtSmem { int self, aux, w0, w1, ident, ones, b0, b1, headw, bar, total; };
template <int D>
__host__ __device__ constexpr EtSmem et_layout() {
  constexpr int KB = D * 2, BLK = kRows * KB;
  EtSmem s{};
  s.self = 0;                          // kNE x [128][KB]             edge-state tiles (TMA in, in-place update, TMA out)
  s.aux = s.self + kNE * BLK;          // kNH x 2 x [128][KB]         h_src | h_dst; hidden overwrites h_src
  s.w0 = s.aux + kNH * 2 * BLK;        // W0 image: 3 K-blocks [D][KB]
  s.w1 = s.w0 + 3 * D * KB;            // W1 image
  s.ident = s.w1 + D * KB;             // identity [D][KB]
  s.ones = s.ident + D * KB;           // [128][32 B]: columns 0..2 = 1.0 (32B swizzle)
  s.b0 = s.ones + kRows * 32;          // [D][32 B]: row n = (hi, mid, lo) of b0[n]
  s.b1 = s.b0 + D * 32;
  s.headw = s.b1 + D * 32;             // fp32 [D]
  s.bar = s.headw + D * 4;
  s.total = s.bar + 256;
  return s;
}

struct EdgeTmaArgs {
  const void* w0_img; const void* w1_img; const void* ident_img; const void* b0_img; const void* b1_img;
  const float* head_w; const float* head_b;
  const __nv_bfloat16* h;
  const int32_t* src; const int32_t* dst;
  const int32_t* n_rows_ptr;
  int max_rows;                // > 0: rows beyond this are not processed (triplet lists are capped at max_triplets)
  float* logit; float* score;
  int do_head;
  int store_e;                 // 0: the new edge state is dead (last step of a plain etx_run: only the classifier reads it)
  int enc;                     // 1: S4b with the paper's input, e0 = MLP([h0_src, h0_dst]) (L133): no old state, K = 2d
};

// all MMAs of one K-block: kbytes of K, 32 bytes (16 bf16) per instruction
template <int KB>
__device__ __forceinline__ void issue_block(uint32_t a_blk, uint32_t b_blk, uint32_t tmem_d, uint32_t idesc) {
#pragma unroll
  for (int s = 0; s < KB / 32; ++s)
    umma::umma<kBf16>(tmem_d, make_desc<KB>(a_blk + s * 32), make_desc<KB>(b_blk + s * 32), idesc, 1u);
}

template <int D>
__global__ void __launch_bounds__(kThreads, 1)
edge_net_tma_kernel(const __grid_constant__ CUtensorMap e_map, const EdgeTmaArgs a) {
  constexpr int KB = D * 2;                                  // bytes per state row = swizzle width
  constexpr int CPR = KB / 16;                               // 16-byte chunks per row
  constexpr int BLK = kRows * KB;
  constexpr EtSmem L = et_layout<D>();
  constexpr uint32_t TMEM_COLS = 8 * D;                      // acc0[2] | acc1[2] | hidden[2] (D/2 packed columns each), pow2
  extern __shared__ uint8_t smem_raw[];
  uint8_t* smem = reinterpret_cast<uint8_t*>((reinterpret_cast<uintptr_t>(smem_raw) + 1023) & ~(uintptr_t)1023);
  float* headw = reinterpret_cast<float*>(smem + L.headw);
  uint64_t* bars = reinterpret_cast<uint64_t*>(smem + L.bar);
  uint64_t *self_full = bars, *self_empty = bars + kNE, *out_ready = bars + 2 * kNE;
  uint64_t *aux_full = bars + 3 * kNE, *aux_empty = aux_full + kNH;
  uint64_t *acc0_full = aux_empty + kNH, *hid_full = acc0_full + 2, *acc1_full = acc0_full + 4, *bar_w = acc0_full + 6;
  uint32_t* tmem_slot = reinterpret_cast<uint32_t*>(acc0_full + 7);

  const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
  const int n_rows = a.max_rows > 0 ? min(*a.n_rows_ptr, a.max_rows) : *a.n_rows_ptr;
  const int n_tiles = (n_rows + kRows - 1) / kRows;

  if (tid == 0) {
    for (int s = 0; s < kNE; ++s) { mbar_init(&self_full[s], 1); mbar_init(&self_empty[s], 1); mbar_init(&out_ready[s], 128); }
    for (int s = 0; s < kNH; ++s) { mbar_init(&aux_full[s], 32); mbar_init(&aux_empty[s], 1); }
    for (int g = 0; g < 2; ++g) { mbar_init(&acc0_full[g], 1); mbar_init(&hid_full[g], 128); mbar_init(&acc1_full[g], 1); }
    mbar_init(bar_w, 1);
    fence_barrier_init();
  }
  if (warp == kMmaWarp) tmem_alloc(tmem_slot, TMEM_COLS);
  for (int i = tid; i < D; i += kThreads) headw[i] = a.head_w[i];
  // the ones tile: row r holds 1.0 in its first three bf16 columns (the three terms of the split bias)
  for (int r = tid; r < kRows; r += kThreads) {
    uint4* row = reinterpret_cast<uint4*>(smem + L.ones + r * 32);
    row[0] = make_uint4(0u, 0u, 0u, 0u); row[1] = make_uint4(0u, 0u, 0u, 0u);
    *reinterpret_cast<uint4*>(smem + L.ones + swz<32>(r, 0)) = make_uint4(0x3f803f80u, 0x00003f80u, 0u, 0u);
  }
  fence_proxy_async();
  tc_fence_before();
  __syncthreads();
  tc_fence_after();
  const uint32_t tmem = *tmem_slot;
  const uint32_t self_addr = smem_u32(smem + L.self), aux_addr = smem_u32(smem + L.aux);

  if (warp >= kEpiWarps && warp < kMmaWarp) {
    // ================================================================================================ gather
    asm volatile("setmaxnreg.dec.sync.aligned.u32 %0;" ::"n"(kGatherRegs));
    // Warp pw < kNH owns slot pw of the gather ring and gathers whole tiles it = pw (mod kNH): wait for the slot,
    // issue the tile's 2 x 128 rows as 16-byte cp.async (64 per lane), wait for them, publish.  Up to kNH tiles are
    // in flight per SM and a tile is published the moment it has landed.  (One warp per slot keeps every waiter at
    // most one mbarrier phase ahead, which the parity wait requires; the warpgroup's fourth warp only donates its
    // registers.)
    const int pw = warp - kEpiWarps;
    for (int it = pw; pw < kNH && blockIdx.x + (long long)it * gridDim.x < n_tiles; it += kNH) {
      const int tile = blockIdx.x + it * gridDim.x;
      const int s = it % kNH;
      int isv[4], idv[4];
#pragma unroll
      for (int j = 0; j < 4; ++j) {
        int row = tile * kRows + j * 32 + lane;
        if (row >= n_rows) row = n_rows - 1;                  // dead rows of the last tile: any valid row
        isv[j] = __ldg(a.src + row); idv[j] = __ldg(a.dst + row);
      }
      mbar_wait(&aux_empty[s], ((it / kNH) & 1) ^ 1);
      const uint32_t st = aux_addr + s * 2 * BLK;
#pragma unroll
      for (int j = 0; j < 4; ++j) {
#pragma unroll
        for (int i = 0; i < CPR; ++i) {
          const int c = i * 32 + lane, rl = c / CPR, piece = c % CPR;
          const int r = j * 32 + rl;
          const int js = __shfl_sync(0xffffffffu, isv[j], rl), jd = __shfl_sync(0xffffffffu, idv[j], rl);
          const uint32_t off = swz<KB>(r, piece);
          cp_async16(st + off, a.h + (size_t)js * D + piece * 8);
          cp_async16(st + BLK + off, a.h + (size_t)jd * D + piece * 8);
        }
      }
      cp_async_commit();
      cp_async_wait<0>();
      fence_proxy_async();                                    // generic-proxy writes -> visible to the tensor core
      mbar_arrive(&aux_full[s]);
    }
  } else if (warp == kLoadWarp) {
    // ================================================================================================ TMA loads
    if (lane == 0) {
      int it = 0;
      for (int tile = blockIdx.x; tile < n_tiles; tile += gridDim.x, ++it) {
        const int s = it % kNE;
        mbar_wait(&self_empty[s], ((it / kNE) & 1) ^ 1);
        if (a.enc) { mbar_arrive(&self_full[s]); continue; }  // no old state: the slot is only the output staging
        mbar_expect_tx(&self_full[s], BLK);
        tma_load_2d(self_addr + s * BLK, &e_map, 0, tile * kRows, &self_full[s]);
      }
    }
  } else if (warp == kStoreWarp) {
    // ================================================================================================ TMA stores
    if (lane == 0) {
      int it = 0;
      for (int tile = blockIdx.x; tile < n_tiles; tile += gridDim.x, ++it) {
        const int s = it % kNE;
        mbar_wait(&out_ready[s], (it / kNE) & 1);
        if (a.store_e) {
          tma_store_2d(&e_map, self_addr + s * BLK, 0, tile * kRows);
          bulk_commit();
          bulk_wait_read0();                                  // the slot has been read: hand it back to the loader
        }
        mbar_arrive(&self_empty[s]);
      }
      bulk_wait0();
    }
  } else if (warp == kMmaWarp) {
    // ================================================================================================ MMA issuer
    if (elect_one()) {
      const uint32_t wb0 = (a.enc ? 2 : 3) * D * KB, wb1 = D * KB, bb = D * 32;
      mbar_expect_tx(bar_w, wb0 + 2 * wb1 + 2 * bb);
      bulk_g2s(smem + L.w0, a.w0_img, wb0, bar_w);
      bulk_g2s(smem + L.w1, a.w1_img, wb1, bar_w);
      bulk_g2s(smem + L.ident, a.ident_img, wb1, bar_w);
      bulk_g2s(smem + L.b0, a.b0_img, bb, bar_w);
      bulk_g2s(smem + L.b1, a.b1_img, bb, bar_w);
      mbar_wait(bar_w, 0);
      const uint32_t idesc = make_idesc<kBf16>(D);
      const uint32_t w0_addr = smem_u32(smem + L.w0), w1_addr = smem_u32(smem + L.w1), id_addr = smem_u32(smem + L.ident);
      const uint64_t ones_desc = make_desc<32>(smem_u32(smem + L.ones));
      const uint64_t b0_desc = make_desc<32>(smem_u32(smem + L.b0)), b1_desc = make_desc<32>(smem_u32(smem + L.b1));
      auto layer1 = [&](int j) {                              // acc1 = 1*b1' + hidden*W1^T + e*I   (tile j of this CTA)
        const int g = j & 1, se = j % kNE;
        mbar_wait(&hid_full[g], (j >> 1) & 1);
        tc_fence_after();
        const uint32_t d1 = tmem + 2 * D + g * D, hid = tmem + 4 * D + g * (D / 2);
        umma::umma<kBf16>(d1, ones_desc, b1_desc, idesc, 0u);
#pragma unroll
        for (int k = 0; k < D / 16; ++k)                      // A = hidden in tensor memory, 8 packed columns per K = 16
          umma_ts(d1, hid + 8 * k, make_desc<KB>(w1_addr + k * 32), idesc, 1u);
        if (!a.enc) issue_block<KB>(self_addr + se * BLK, id_addr, d1, idesc);             // + old e (R14)
        umma_commit(&acc1_full[g]);
      };
      // Issue order: layer 0 of tile it, then layer 1 of tile it-1 (so the tensor pipe always has the next tile's
      // big layer queued) -- but while tile it's operands are still in flight, a layer 1 that has become ready
      // is issued first instead of waiting behind them.
      int it = 0, pending = -1;                               // pending: tile whose layer 1 has not been issued yet
      for (int tile = blockIdx.x; tile < n_tiles; tile += gridDim.x, ++it) {
        const int g = it & 1, se = it % kNE, sh = it % kNH;
        for (uint32_t spins = 0;; ++spins) {
          if (pending >= 0 && mbar_test(&hid_full[pending & 1], (pending >> 1) & 1)) { layer1(pending); pending = -1; }
          if (mbar_test(&aux_full[sh], (it / kNH) & 1) && mbar_test(&self_full[se], (it / kNE) & 1)) break;
          if ((spins & 0xfffffu) == 0xfffffu && mbar_stalled(spins)) __trap();
        }
        tc_fence_after();
        // acc0[g] was drained by epilogue 0 of tile it-2: hid_full, waited on for layer 1 of it-2, covers it
        const uint32_t d0 = tmem + g * D;
        umma::umma<kBf16>(d0, ones_desc, b0_desc, idesc, 0u);
        issue_block<KB>(aux_addr + sh * 2 * BLK, w0_addr, d0, idesc);                      // h_src
        issue_block<KB>(aux_addr + sh * 2 * BLK + BLK, w0_addr + D * KB, d0, idesc);       // h_dst
        if (!a.enc) issue_block<KB>(self_addr + se * BLK, w0_addr + 2 * D * KB, d0, idesc);   // e
        umma_commit(&acc0_full[g]);
        umma_commit(&aux_empty[sh]);                          // layer 0 was the gather slot's only reader
        if (pending >= 0) layer1(pending);
        pending = it;
      }
      if (pending >= 0) layer1(pending);
    }
  } else {
    // ================================================================================================ epilogue
    asm volatile("setmaxnreg.inc.sync.aligned.u32 %0;" ::"n"(kEpiRegs));
    const int g = warp >> 2, q = warp & 3;                    // warpgroup, TMEM lane quarter
    const int r = q * 32 + lane;                              // row of the tile owned by this thread
    const uint32_t lane_base = (uint32_t)(q * 32) << 16;
    const float head_b = a.head_b[0];
    int j = 0;
    for (int it = g; blockIdx.x + (long long)it * gridDim.x < n_tiles; it += 2, ++j) {
      const int tile = blockIdx.x + it * gridDim.x;
      const int row = tile * kRows + r;
      uint8_t* out = smem + L.self + (it % kNE) * BLK;        // the e tile, updated in place
      // ---- epilogue 0: relu(acc0) -> bf16, packed two per column -> tensor memory, the A operand of layer 1 (R3, R20);
      //      the bias is already in acc0
      mbar_wait(&acc0_full[g], j & 1);
      tc_fence_after();
#pragma unroll
      for (int c0 = 0; c0 < D; c0 += 64) {
        uint32_t v[32], w[32], pk[32];
        tmem_ld32_nowait(tmem + lane_base + g * D + c0, v);
        if (D > 32) tmem_ld32_nowait(tmem + lane_base + g * D + c0 + 32, w);
        tmem_ld_wait();
#pragma unroll
        for (int i = 0; i < 16; ++i) pk[i] = pack_bf16x2_relu(__uint_as_float(v[2 * i]), __uint_as_float(v[2 * i + 1]));
        if (D > 32) {
#pragma unroll
          for (int i = 0; i < 16; ++i) pk[16 + i] = pack_bf16x2_relu(__uint_as_float(w[2 * i]), __uint_as_float(w[2 * i + 1]));
          tmem_st32(tmem + lane_base + 4 * D + g * (D / 2) + c0 / 2, pk);
        } else {
          tmem_st16(tmem + lane_base + 4 * D + g * (D / 2), pk);
        }
      }
      tmem_st_wait();
      tc_fence_before();
      mbar_arrive(&hid_full[g]);
      // ---- epilogue 1: acc1 (= b1 + W1 hidden + old e) -> bf16 -> the slot, optional classifier (R14, R16, R20)
      mbar_wait(&acc1_full[g], j & 1);
      tc_fence_after();
      float hacc = 0.0f;
#pragma unroll
      for (int c0 = 0; c0 < D; c0 += 32) {
        uint32_t v[32];
        tmem_ld32_nowait(tmem + lane_base + 2 * D + g * D + c0, v);
        tmem_ld_wait();
#pragma unroll
        for (int ch = 0; ch < 4; ++ch) {
          uint4 qv;
          qv.x = pack_bf16x2(__uint_as_float(v[ch * 8 + 0]), __uint_as_float(v[ch * 8 + 1]));
          qv.y = pack_bf16x2(__uint_as_float(v[ch * 8 + 2]), __uint_as_float(v[ch * 8 + 3]));
          qv.z = pack_bf16x2(__uint_as_float(v[ch * 8 + 4]), __uint_as_float(v[ch * 8 + 5]));
          qv.w = pack_bf16x2(__uint_as_float(v[ch * 8 + 6]), __uint_as_float(v[ch * 8 + 7]));
          if (a.store_e) *reinterpret_cast<uint4*>(out + swz<KB>(r, c0 / 8 + ch)) = qv;
          if (a.do_head) {                                    // the classifier sees the stored bf16 state, ascending j
            const float* hw = headw + c0 + ch * 8;
            hacc = __fmaf_rn(bf16_lo(qv.x), hw[0], hacc); hacc = __fmaf_rn(bf16_hi(qv.x), hw[1], hacc);
            hacc = __fmaf_rn(bf16_lo(qv.y), hw[2], hacc); hacc = __fmaf_rn(bf16_hi(qv.y), hw[3], hacc);
            hacc = __fmaf_rn(bf16_lo(qv.z), hw[4], hacc); hacc = __fmaf_rn(bf16_hi(qv.z), hw[5], hacc);
            hacc = __fmaf_rn(bf16_lo(qv.w), hw[6], hacc); hacc = __fmaf_rn(bf16_hi(qv.w), hw[7], hacc);
          }
        }
      }
      tc_fence_before();                                      // acc1[g] may be overwritten after our next hid_full arrive
      fence_proxy_async();                                    // generic-proxy writes -> visible to the TMA store
      mbar_arrive(&out_ready[it % kNE]);
      if (a.do_head && row < n_rows) {
        const float z = __fadd_rn(hacc, head_b);
        a.logit[row] = z;
        a.score[row] = 1.0f / (1.0f + expf(-z));
      }
    }
  }
  tc_fence_before();
  __syncthreads();
  if (warp == kMmaWarp) tmem_dealloc(tmem, TMEM_COLS);
}

// ---------------------------------------------------------------------------------------------- S4b edge encoder
// e0 = W1 relu(W0 |f_dst - f_src| + b0) + b1  (PAPER.md L133 with the configs' K = 3 input, R10 / R11).
// The stage only WRITES the edge state (E * d * 2 bytes), so it is bound by that write plus the FFMA work of the
// K = 3 layer, which stays on the fp32 pipe in the pinned order (R3, R20).  Five warpgroups each own the CTA's
// tiles it = w (mod 5) from front to back (five is what tensor memory holds: 5 x (D + D/2) = 480 of 512 columns): gather the two feature rows (prefetched one tile ahead, their indices
// two tiles ahead), layer 0 on the FFMA pipe, relu -> bf16 -> tensor memory (the A operand of layer 1), wait for
// the MMA, TMEM -> bf16 -> the warpgroup's swizzled shared-memory slot, and one TMA store per tile.
constexpr int kEncGroups = 5;
constexpr int kEncMmaWarp = kEncGroups * 4, kEncStoreWarp = kEncMmaWarp + 1;
constexpr int kEncThreads = (kEncStoreWarp + 1) * 32;      // 704

struct EncSmem { int out, w1, ones, b1, w3, bar, total; };
template <int D>
__host__ __device__ constexpr EncSmem enc_layout() {
  constexpr int KB = D * 2, BLK = kRows * KB;
  EncSmem s{};
  s.out = 0;                           // 2 x kEncGroups x [128][KB] output staging (two slots per warpgroup)
  s.w1 = s.out + 2 * kEncGroups * BLK; // W1 image [D][KB]
  s.ones = s.w1 + D * KB;              // [128][32 B]
  s.b1 = s.ones + kRows * 32;          // [D][32 B] split bias of layer 1
  s.w3 = s.b1 + D * 32;                // fp32: W0^T [3][D], b0 [D]
  s.bar = s.w3 + 4 * D * 4;
  s.total = s.bar + 256;
  return s;
}

struct EdgeEncArgs {
  const void* w1_img; const void* b1_img;
  float w0t[3 * 64];         // [3][D] fp32 (W0 transposed) and b0[D], passed BY VALUE: kernel parameters live in the
  float b0[64];              // constant bank, so the FFMAs of layer 0 take them as operands without any load
  const float4* feat;
  const int32_t* src; const int32_t* dst;
  const int32_t* n_rows_ptr; // edge encoder: E on the device
  int n_rows;                // node encoder (S4a): number of hits
  int node;                  // 1: h0 = MLP(f) over hits, rows are the hits themselves; 0: e0 = MLP(|f_dst - f_src|) over edges
};

template <int D>
__global__ void __launch_bounds__(kEncThreads, 1)
edge_enc_tma_kernel(const __grid_constant__ CUtensorMap e_map, const EdgeEncArgs a) {
  constexpr int KB = D * 2, BLK = kRows * KB;
  constexpr EncSmem L = enc_layout<D>();
  constexpr uint32_t TMEM_COLS = 8 * D;                      // acc[5] (D each) | hidden[5] (D/2 each) = 7.5 D, pow2
  extern __shared__ uint8_t smem_raw[];
  uint8_t* smem = reinterpret_cast<uint8_t*>((reinterpret_cast<uintptr_t>(smem_raw) + 1023) & ~(uintptr_t)1023);
  uint64_t* bars = reinterpret_cast<uint64_t*>(smem + L.bar);
  uint64_t *hid_full = bars, *acc_full = bars + kEncGroups, *out_ready = bars + 2 * kEncGroups,
           *slot_free = bars + 4 * kEncGroups, *bar_w = bars + 6 * kEncGroups;
  uint32_t* tmem_slot = reinterpret_cast<uint32_t*>(bar_w + 1);

  const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
  const int n_rows = a.node ? a.n_rows : *a.n_rows_ptr;
  const int n_tiles = (n_rows + kRows - 1) / kRows;

  if (tid == 0) {
    for (int g = 0; g < kEncGroups; ++g) {
      mbar_init(&hid_full[g], 128); mbar_init(&acc_full[g], 1);
      for (int b = 0; b < 2; ++b) { mbar_init(&out_ready[2 * g + b], 128); mbar_init(&slot_free[2 * g + b], 1); }
    }
    mbar_init(bar_w, 1);
    fence_barrier_init();
  }
  if (warp == kEncMmaWarp) tmem_alloc(tmem_slot, TMEM_COLS);
  for (int r = tid; r < kRows; r += kEncThreads) {
    uint4* row = reinterpret_cast<uint4*>(smem + L.ones + r * 32);
    row[0] = make_uint4(0u, 0u, 0u, 0u); row[1] = make_uint4(0u, 0u, 0u, 0u);
    *reinterpret_cast<uint4*>(smem + L.ones + swz<32>(r, 0)) = make_uint4(0x3f803f80u, 0x00003f80u, 0u, 0u);
  }
  fence_proxy_async();
  tc_fence_before();
  __syncthreads();
  tc_fence_after();
  const uint32_t tmem = *tmem_slot;
  const uint32_t out_addr = smem_u32(smem + L.out);

  if (warp == kEncStoreWarp) {
    // ================================================================================================ TMA stores
    // One TMA store per tile.  (Measured alternatives, both without gain: two stores in flight per SM -- the stage
    // stays at 0.34 ms, the TMA unit reads a 16 KB tile out of shared memory at ~17 bytes per cycle whatever the depth;
    // the store warp copying the tile out with 16-byte plain stores -- 1.02 ms.)
    if (lane == 0) {
      int it = 0;
      for (int tile = blockIdx.x; tile < n_tiles; tile += gridDim.x, ++it) {
        const int g = it % kEncGroups;
        const int jj = it / kEncGroups, sl = 2 * g + (jj & 1);  // the group's tiles alternate between its two slots
        mbar_wait(&out_ready[sl], (jj >> 1) & 1);
        tma_store_2d(&e_map, out_addr + sl * BLK, 0, tile * kRows);
        bulk_commit();
        bulk_wait_read0();
        mbar_arrive(&slot_free[sl]);
      }
      bulk_wait0();
    }
  } else if (warp == kEncMmaWarp) {
    // ================================================================================================ MMA issuer
    if (elect_one()) {
      const uint32_t wb1 = D * KB, bb = D * 32;
      mbar_expect_tx(bar_w, wb1 + bb);
      bulk_g2s(smem + L.w1, a.w1_img, wb1, bar_w);
      bulk_g2s(smem + L.b1, a.b1_img, bb, bar_w);
      mbar_wait(bar_w, 0);
      const uint32_t idesc = make_idesc<kBf16>(D);
      const uint32_t w1_addr = smem_u32(smem + L.w1);
      const uint64_t ones_desc = make_desc<32>(smem_u32(smem + L.ones)), b1_desc = make_desc<32>(smem_u32(smem + L.b1));
      int it = 0;
      for (int tile = blockIdx.x; tile < n_tiles; tile += gridDim.x, ++it) {
        const int g = it % kEncGroups;
        mbar_wait(&hid_full[g], (it / kEncGroups) & 1);       // also: the group has drained acc[g] of its last tile
        tc_fence_after();
        const uint32_t d1 = tmem + g * D, hid = tmem + kEncGroups * D + g * (D / 2);
        umma::umma<kBf16>(d1, ones_desc, b1_desc, idesc, 0u);
#pragma unroll
        for (int k = 0; k < D / 16; ++k) umma_ts(d1, hid + 8 * k, make_desc<KB>(w1_addr + k * 32), idesc, 1u);
        umma_commit(&acc_full[g]);
      }
    }
  } else {
    // ================================================================================================ compute groups
    const int g = warp >> 2, q = warp & 3;
    const int r = q * 32 + lane;                              // row of the tile owned by this thread
    const uint32_t lane_base = (uint32_t)(q * 32) << 16;
    auto tile_of = [&](int j) { return blockIdx.x + (long long)(g + j * kEncGroups) * gridDim.x; };
    auto load_idx = [&](int j, int& is, int& id) {
      const long long t = tile_of(j);
      is = 0; id = 0;
      if (t < n_tiles) {
        long long row = t * kRows + r;
        if (row >= n_rows) row = n_rows - 1;
        if (a.node) { is = (int)row; id = (int)row; }
        else { is = __ldg(a.src + row); id = __ldg(a.dst + row); }
      }
    };
    int is_n, id_n;                                           // indices of tile j + 1
    float4 fs, fd;                                            // features of tile j
    {
      int is0, id0;
      load_idx(0, is0, id0);
      load_idx(1, is_n, id_n);
      fs = __ldg(a.feat + is0); fd = __ldg(a.feat + id0);
    }
    for (int j = 0; tile_of(j) < n_tiles; ++j) {
      const long long tile = tile_of(j);
      // R11: component-wise |f_dst - f_src| of the normalised features
      float fx = fabsf(__fsub_rn(fd.x, fs.x)), fy = fabsf(__fsub_rn(fd.y, fs.y)), fz = fabsf(__fsub_rn(fd.z, fs.z));
      if (a.node) { fx = fs.x; fy = fs.y; fz = fs.z; }        // S4a: the hit's own normalised features
      // prefetch: features of tile j + 1 (their indices are here), indices of tile j + 2
      fs = __ldg(a.feat + is_n); fd = __ldg(a.feat + id_n);
      load_idx(j + 2, is_n, id_n);
      // ---- layer 0 on the FFMA pipe, pinned order (R3); relu -> bf16 -> tensor memory
#pragma unroll
      for (int c0 = 0; c0 < D; c0 += 64) {
        uint32_t pk[32];
#pragma unroll
        for (int i = 0; i < (D > 32 ? 32 : 16); ++i) {
          float y[2];
#pragma unroll
          for (int h = 0; h < 2; ++h) {
            const int c = c0 + 2 * i + h;
            float acc = __fmaf_rn(fx, a.w0t[c], 0.0f);
            acc = __fmaf_rn(fy, a.w0t[D + c], acc);
            acc = __fmaf_rn(fz, a.w0t[2 * D + c], acc);
            y[h] = __fadd_rn(acc, a.b0[c]);
          }
          pk[i] = pack_bf16x2_relu(y[0], y[1]);
        }
        if (D > 32) tmem_st32(tmem + lane_base + kEncGroups * D + g * (D / 2) + c0 / 2, pk);
        else tmem_st16(tmem + lane_base + kEncGroups * D + g * (D / 2), pk);
      }
      tmem_st_wait();
      tc_fence_before();
      mbar_arrive(&hid_full[g]);
      // ---- layer 1 result (bias already inside): TMEM -> bf16 -> the group's slot -> TMA store (R20)
      const int sl = 2 * g + (j & 1);
      uint8_t* out = smem + L.out + sl * BLK;
      mbar_wait(&slot_free[sl], ((j >> 1) & 1) ^ 1);          // the store of tile j - 2 has read the slot
      mbar_wait(&acc_full[g], j & 1);
      tc_fence_after();
#pragma unroll
      for (int c0 = 0; c0 < D; c0 += 32) {
        uint32_t v[32];
        tmem_ld32_nowait(tmem + lane_base + g * D + c0, v);
        tmem_ld_wait();
#pragma unroll
        for (int ch = 0; ch < 4; ++ch) {
          uint4 qv;
          qv.x = pack_bf16x2(__uint_as_float(v[ch * 8 + 0]), __uint_as_float(v[ch * 8 + 1]));
          qv.y = pack_bf16x2(__uint_as_float(v[ch * 8 + 2]), __uint_as_float(v[ch * 8 + 3]));
          qv.z = pack_bf16x2(__uint_as_float(v[ch * 8 + 4]), __uint_as_float(v[ch * 8 + 5]));
          qv.w = pack_bf16x2(__uint_as_float(v[ch * 8 + 6]), __uint_as_float(v[ch * 8 + 7]));
          *reinterpret_cast<uint4*>(out + swz<KB>(r, c0 / 8 + ch)) = qv;
        }
      }
      tc_fence_before();
      fence_proxy_async();
      mbar_arrive(&out_ready[sl]);
      (void)tile;
    }
  }
  tc_fence_before();
  __syncthreads();
  if (warp == kEncMmaWarp) tmem_dealloc(tmem, TMEM_COLS);
}

// ---------------------------------------------------------------------------------------------- host side
uint16_t bf16_bits_rne(float x) {
  const __nv_bfloat16 b = __float2bfloat16_rn(x);
  uint16_t u; memcpy(&u, &b, 2);
  return u;
}
float bf16_value(uint16_t u) { uint32_t w = (uint32_t)u << 16; float f; memcpy(&f, &w, 4); return f; }

// [n][32 B] image (32B swizzle) whose row n holds, in its first three bf16 columns, an exact split of v[n]:
// hi = rn(v), mid = rn(v - hi), lo = v - hi - mid (at most 8 significant bits are left, so lo is exact)
std::vector<uint8_t> pack_split_rows(const std::vector<float>& v) {
  const int n = (int)v.size();
  std::vector<uint8_t> img((size_t)n * 32, 0);
  for (int r = 0; r < n; ++r) {
    float rest = v[r];
    uint16_t t[3];
    for (int i = 0; i < 3; ++i) { t[i] = bf16_bits_rne(rest); rest -= bf16_value(t[i]); }
    const uint32_t lin = (uint32_t)r * 32;
    const size_t off = lin + ((((lin >> 7)) & 1u) << 4);      // chunk 0 of the row under the 32B swizzle
    memcpy(&img[off], t, 6);
  }
  return img;
}

// identity [D][KB] in the K-major swizzled operand layout (row n has 1.0 at column n)
std::vector<uint8_t> pack_identity(int D) {
  const int KB = D * 2;
  std::vector<uint8_t> img((size_t)D * KB, 0);
  for (int n = 0; n < D; ++n) {
    const int b = n * 2, chunk = b / 16;
    const uint32_t lin = (uint32_t)n * KB;
    const size_t off = lin + (((chunk ^ (lin >> 7)) & (KB / 16 - 1)) << 4) + (b & 15);
    img[off] = 0x80; img[off + 1] = 0x3f;
  }
  return img;
}

void* upload_bytes(etx_ctx* c, const std::vector<uint8_t>& v) {
  void* p = etx_device_alloc(c, v.size());
  if (!p) return nullptr;
  cudaMemcpy(p, v.data(), v.size(), cudaMemcpyHostToDevice);
  return p;
}

typedef CUresult (*EncodeTiledFn)(CUtensorMap*, CUtensorMapDataType, cuuint32_t, void*, const cuuint64_t*, const cuuint64_t*,
                                  const cuuint32_t*, const cuuint32_t*, CUtensorMapInterleave, CUtensorMapSwizzle,
                                  CUtensorMapL2promotion, CUtensorMapFloatOOBfill);

template <int D>
void edge_tma_launch(etx_ctx* c, const EdgeTmaArgs& a, int max_rows, cudaStream_t s) {
  auto kern = edge_net_tma_kernel<D>;
  constexpr int smem = et_layout<D>().total + 1024;
  opt_in_smem(c, kern, smem);
  const int tiles = (max_rows + kRows - 1) / kRows;
  const int grid = tiles < c->sm_count ? tiles : c->sm_count;     // one persistent CTA per SM
  if (grid <= 0) return;
  CUtensorMap map;
  memcpy(&map, c->e_map, sizeof(map));
  kern<<<grid, kThreads, smem, s>>>(map, a);
  c->launches++;
}

template <int D>
void edge_enc_launch(etx_ctx* c, const EdgeEncArgs& a, const unsigned char* out_map, int max_rows, cudaStream_t s) {
  auto kern = edge_enc_tma_kernel<D>;
  constexpr int smem = enc_layout<D>().total + 1024;
  opt_in_smem(c, kern, smem);
  const int tiles = (max_rows + kRows - 1) / kRows;
  const int grid = tiles < c->sm_count ? tiles : c->sm_count;     // one persistent CTA per SM (512 TMEM columns)
  if (grid <= 0) return;
  CUtensorMap map;
  memcpy(&map, out_map, sizeof(map));
  kern<<<grid, kEncThreads, smem, s>>>(map, a);
  c->launches++;
}

}  // namespace

// bf16 mode, tensor engine: per-step bias / identity images and the tensor map of the edge state
bool edge_tma_configure(etx_ctx* c) {
  const int D = c->hp.gnn_latent, L = c->hp.gnn_iters;
  static_assert(sizeof(CUtensorMap) == sizeof(c->e_map), "etx_ctx::e_map must hold a CUtensorMap");
  c->ident_img = upload_bytes(c, pack_identity(D));
  if (!c->ident_img) return false;
  c->edge_bias_img.assign(2 * (size_t)L, nullptr);
  for (int it = 0; it < L; ++it)
    for (int l = 0; l < 2; ++l) {
      void* p = upload_bytes(c, pack_split_rows(c->layers[c->i_iter0 + 4 * it + 2 + l].b));
      if (!p) return false;
      c->edge_bias_img[2 * it + l] = p;
    }
  c->eenc_b0_img = upload_bytes(c, pack_split_rows(c->layers[c->i_eenc].b));
  if (!c->eenc_b0_img) return false;
  c->eenc_b1_img = upload_bytes(c, pack_split_rows(c->layers[c->i_eenc + 1].b));
  c->nenc_b1_img = upload_bytes(c, pack_split_rows(c->layers[c->i_nenc + 1].b));
  if (!c->eenc_b1_img || !c->nenc_b1_img) return false;
  if (c->i_trip >= 0) {
    c->trip_b0_img[0] = upload_bytes(c, pack_split_rows(c->layers[c->i_trip].b));
    c->trip_b0_img[1] = upload_bytes(c, pack_split_rows(c->layers[c->i_trip + 2].b));
    c->zero_bias_img = upload_bytes(c, pack_split_rows(std::vector<float>((size_t)D, 0.0f)));
    if (!c->trip_b0_img[0] || !c->trip_b0_img[1] || !c->zero_bias_img) return false;
  }
  void* fn = nullptr;
  cudaDriverEntryPointQueryResult qres;
  if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &fn, cudaEnableDefault, &qres) != cudaSuccess || !fn) return false;
  const cuuint64_t rows = c->max_edges > 0 ? (cuuint64_t)c->max_edges : 1;
  const cuuint64_t gdim[2] = {(cuuint64_t)D, rows};
  const cuuint64_t gstride[1] = {(cuuint64_t)D * 2};
  const cuuint32_t box[2] = {(cuuint32_t)D, (cuuint32_t)kRows};
  const cuuint32_t estr[2] = {1, 1};
  CUtensorMap map;
  const CUresult r = reinterpret_cast<EncodeTiledFn>(fn)(
      &map, CU_TENSOR_MAP_DATA_TYPE_BFLOAT16, 2, c->e, gdim, gstride, box, estr, CU_TENSOR_MAP_INTERLEAVE_NONE,
      D == 64 ? CU_TENSOR_MAP_SWIZZLE_128B : CU_TENSOR_MAP_SWIZZLE_64B, CU_TENSOR_MAP_L2_PROMOTION_L2_256B,
      CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
  if (r != CUDA_SUCCESS) return false;
  memcpy(c->e_map, &map, sizeof(map));
  const cuuint64_t hdim[2] = {(cuuint64_t)D, c->hp.max_hits > 0 ? (cuuint64_t)c->hp.max_hits : 1};
  const CUresult r2 = reinterpret_cast<EncodeTiledFn>(fn)(
      &map, CU_TENSOR_MAP_DATA_TYPE_BFLOAT16, 2, c->h, hdim, gstride, box, estr, CU_TENSOR_MAP_INTERLEAVE_NONE,
      D == 64 ? CU_TENSOR_MAP_SWIZZLE_128B : CU_TENSOR_MAP_SWIZZLE_64B, CU_TENSOR_MAP_L2_PROMOTION_L2_256B,
      CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
  if (r2 != CUDA_SUCCESS) return false;
  memcpy(c->h_map, &map, sizeof(map));
  return true;
}

void launch_edge_net_tma(etx_ctx* c, int iter, int n_hits, bool do_head, cudaStream_t s) {
  const int i0 = c->i_iter0 + 4 * iter + 2;
  EdgeTmaArgs a;
  a.w0_img = c->layers[i0].dev.Wtc; a.w1_img = c->layers[i0 + 1].dev.Wtc; a.ident_img = c->ident_img;
  a.b0_img = c->edge_bias_img[2 * iter]; a.b1_img = c->edge_bias_img[2 * iter + 1];
  a.head_w = c->layers[c->i_head].dev.Wt; a.head_b = c->layers[c->i_head].dev.bias;
  a.h = static_cast<const __nv_bfloat16*>(c->h);
  a.src = c->src; a.dst = c->dst; a.n_rows_ptr = c->n_edges;
  a.logit = c->logit; a.score = c->score_out; a.do_head = do_head ? 1 : 0;
  a.store_e = (do_head && !c->keep_final_state) ? 0 : 1;
  a.enc = 0; a.max_rows = 0;
  const long long max_rows_ll = (long long)n_hits * c->hp.k;
  const int max_rows = (int)(max_rows_ll > 0x7fffffff ? 0x7fffffff : max_rows_ll);
  if (c->hp.gnn_latent == 32) edge_tma_launch<32>(c, a, max_rows, s);
  else edge_tma_launch<64>(c, a, max_rows, s);
}

// S4b with the paper's edge-encoder input (edge_enc_input == 1, L133): e0 = MLP([h0_src, h0_dst]).  The edge-network kernel
// without an old state: nothing is loaded into the state slots, layer 0 has two K-blocks, layer 1 no identity block.
void launch_edge_enc_h_tma(etx_ctx* c, int n_hits, bool do_head, cudaStream_t s) {
  const int i0 = c->i_eenc;
  EdgeTmaArgs a;
  a.w0_img = c->layers[i0].dev.Wtc; a.w1_img = c->layers[i0 + 1].dev.Wtc; a.ident_img = c->ident_img;
  a.b0_img = c->eenc_b0_img; a.b1_img = c->eenc_b1_img;
  a.head_w = c->layers[c->i_head].dev.Wt; a.head_b = c->layers[c->i_head].dev.bias;
  a.h = static_cast<const __nv_bfloat16*>(c->h);
  a.src = c->src; a.dst = c->dst; a.n_rows_ptr = c->n_edges;
  a.logit = c->logit; a.score = c->score_out; a.do_head = do_head ? 1 : 0;
  a.store_e = 1; a.enc = 1; a.max_rows = 0;
  const long long max_rows_ll = (long long)n_hits * c->hp.k;
  const int max_rows = (int)(max_rows_ll > 0x7fffffff ? 0x7fffffff : max_rows_ll);
  if (c->hp.gnn_latent == 32) edge_tma_launch<32>(c, a, max_rows, s);
  else edge_tma_launch<64>(c, a, max_rows, s);
}

// Triplet classifier (R28) on the tensor cores: the edge-network kernel in its
// no-old-state mode gathers the two final edge encodings of a triplet (rows of e, by the triplet's edge ids) as the two
// K-blocks of layer 0 (W0 = the classifier's 2d -> d layer, bias inside the MMA), rounds relu(acc0) to bf16 -- R20's
// operand rounding -- and runs a "layer 1" whose weight is the identity and whose bias is zero, which hands the bf16
// hidden activations through exactly; the fused head then IS the classifier's d -> 1 layer: an fp32 chain in ascending
// j over the bf16 hidden values, plus bias, and the sigmoid.  Nothing is stored but logit and score.
void launch_triplet_cls_tma(etx_ctx* c, int kind, cudaStream_t s) {
  const int i0 = c->i_trip + (kind ? 2 : 0);
  const size_t cap = (size_t)c->hp.max_triplets;
  EdgeTmaArgs a;
  a.w0_img = c->layers[i0].dev.Wtc; a.w1_img = c->ident_img; a.ident_img = c->ident_img;
  a.b0_img = c->trip_b0_img[kind ? 1 : 0]; a.b1_img = c->zero_bias_img;
  a.head_w = c->layers[i0 + 1].dev.Wt; a.head_b = c->layers[i0 + 1].dev.bias;
  a.h = static_cast<const __nv_bfloat16*>(c->e);
  a.src = c->trip_first + kind * cap; a.dst = c->trip_second + kind * cap;
  a.n_rows_ptr = c->trip_total + kind; a.max_rows = c->hp.max_triplets;
  a.logit = c->trip_logit + kind * cap; a.score = c->trip_score + kind * cap;
  a.do_head = 1; a.store_e = 0; a.enc = 1;
  if (c->hp.gnn_latent == 32) edge_tma_launch<32>(c, a, c->hp.max_triplets, s);
  else edge_tma_launch<64>(c, a, c->hp.max_triplets, s);
}

// S4b with the configs' K = 3 edge-encoder input (edge_enc_input == 0), or S4a (node = true): the same kernel over hits
void launch_edge_enc_tma(etx_ctx* c, int n_hits, bool node, cudaStream_t s) {
  const int i0 = node ? c->i_nenc : c->i_eenc;
  EdgeEncArgs a;
  a.w1_img = c->layers[i0 + 1].dev.Wtc; a.b1_img = node ? c->nenc_b1_img : c->eenc_b1_img;
  const int D = c->hp.gnn_latent;                            // 32 or 64 (umma_supported)
  for (int n = 0; n < D; ++n) {
    for (int k = 0; k < 3; ++k) a.w0t[k * D + n] = c->layers[i0].W[(size_t)n * 3 + k];
    a.b0[n] = c->layers[i0].b[n];
  }
  a.feat = c->feat; a.src = c->src; a.dst = c->dst; a.n_rows_ptr = c->n_edges;
  a.n_rows = n_hits; a.node = node ? 1 : 0;
  const long long max_rows_ll = node ? (long long)n_hits : (long long)n_hits * c->hp.k;
  const int max_rows = (int)(max_rows_ll > 0x7fffffff ? 0x7fffffff : max_rows_ll);
  const unsigned char* map = node ? c->h_map : c->e_map;
  if (c->hp.gnn_latent == 32) edge_enc_launch<32>(c, a, map, max_rows, s);
  else edge_enc_launch<64>(c, a, map, max_rows, s);
}

}  // namespace etx
