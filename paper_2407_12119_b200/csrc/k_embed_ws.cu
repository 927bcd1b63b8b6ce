// S1, bf16 mode: the hit-embedding MLP  emb = W_H relu(... relu(W_0 f + b_0) ...) + b_H  (sec. 5.1;
// shapes from the configs, R2: 3 -> D -> ... -> D -> 4 with D = 64 or 128 and two or three hidden layers).
//
// 67 kFLOP per hit and 32 bytes of HBM traffic: the stage is bound by the tensor pipe and by the epilogue ALU work,
// never by memory, so the kernel is organised to keep both busy.  One persistent CTA per SM; four warpgroups each
// take a 128-hit tile from its features to its embedding (layer 0, K = 3, on the FFMA pipe in the pinned order with
// its weights as kernel parameters, i.e. constant-bank operands; every epilogue: TMEM -> + bias -> relu -> bf16 ->
// the tile's swizzled A operand in shared memory, rewritten in place); a fifth role, one elected thread, issues the
// tcgen05.mma of whichever warpgroup has an operand ready.  The weights of the tensor layers are brought in once
// per CTA (cp.async.bulk) and shared by the four warpgroups; accumulators live in tensor memory (D columns per
// warpgroup, the 16-column output layer reuses them).  With four tiles in flight per SM the MMAs of one warpgroup
// run under the epilogues of the others; the serial one-tile-per-CTA kernel this replaces (embed_umma_kernel, still
// used for INT8 and for deeper embeddings) left both pipes idle most of the time.
//
// Arithmetic and rounding points are those of embed_umma_kernel (R3, R20): layer 0 in fp32 with ascending-k fmaf,
// hidden activations rounded to bf16 (RNE), fp32 accumulation, bias added in fp32, fp32 output.
#include "umma_common.cuh"

namespace etx {

namespace {

using namespace umma;

constexpr int kEmbGroups = 4;
constexpr int kEmbMmaWarp = kEmbGroups * 4;
constexpr int kEmbThreads = (kEmbMmaWarp + 1) * 32;       // 544
constexpr int kEmbMaxMid = 2;                              // D -> D tensor layers held in shared memory / parameters
constexpr int kEmbBlk = kRows * 128;                       // one K-block of an operand tile: [128 rows][128 B]

struct EmbWsArgs {
  float w0t[3 * 128];        // layer 0: W^T [3][D]                      -- passed BY VALUE: kernel parameters live in the
  float b0[128];             //          b [D]                              constant bank, so the FFMAs and bias adds take
  float bmid[kEmbMaxMid][128];   // biases of the D -> D layers              them as operands without any load
  float bout[4];             // bias of the D -> 4 layer
  const void* wmid_img[kEmbMaxMid];   // [D/64 K-blocks][D rows][128 B] swizzled bf16 images (umma_configure)
  const void* wout_img;      // [D/64][16][128 B]
  const float4* feat;
  float4* emb;
  int n_rows, n_mid;
};

template <int D>
__host__ __device__ constexpr int emb_ws_smem(int n_mid) {
  return kEmbGroups * kRows * D * 2 + n_mid * D * D * 2 + 16 * D * 2 + 128;
}

// bf16x2 words of 32 consecutive activations -> row r of an operand tile, columns c0 .. c0+31
__device__ __forceinline__ void store_row32(uint8_t* tile, uint32_t r, int c0, const uint32_t (&pk)[16]) {
#pragma unroll
  for (int ch = 0; ch < 4; ++ch) {
    const int chunk = c0 / 8 + ch;                           // 16-byte chunk of the row
    *reinterpret_cast<uint4*>(tile + (chunk >> 3) * kEmbBlk + swz<128>(r, chunk & 7)) =
        make_uint4(pk[4 * ch], pk[4 * ch + 1], pk[4 * ch + 2], pk[4 * ch + 3]);
  }
}

template <int D>
__global__ void __launch_bounds__(kEmbThreads, 1) embed_ws_kernel(const EmbWsArgs a) {
  constexpr int ROWB = D * 2;                                // bytes per activation row
  constexpr int TILE = kRows * ROWB;                         // one warpgroup's operand tile
  constexpr uint32_t TMEM_COLS = kEmbGroups * D;             // 512 (D = 128) or 256 (D = 64)
  extern __shared__ uint8_t smem_raw[];
  uint8_t* smem = reinterpret_cast<uint8_t*>((reinterpret_cast<uintptr_t>(smem_raw) + 1023) & ~(uintptr_t)1023);
  uint8_t* A = smem;
  uint8_t* W = A + kEmbGroups * TILE;
  const int n_mid = a.n_mid, H = n_mid + 1;                  // tensor layers per tile
  uint64_t* bars = reinterpret_cast<uint64_t*>(W + n_mid * D * ROWB + 16 * ROWB);
  uint64_t *a_ready = bars, *acc_full = bars + kEmbGroups, *bar_w = bars + 2 * kEmbGroups;
  uint32_t* tmem_slot = reinterpret_cast<uint32_t*>(bar_w + 1);

  const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
  const int n_tiles = (a.n_rows + kRows - 1) / kRows;

  if (tid == 0) {
    for (int g = 0; g < kEmbGroups; ++g) { mbar_init(&a_ready[g], 128); mbar_init(&acc_full[g], 1); }
    mbar_init(bar_w, 1);
    fence_barrier_init();
  }
  if (warp == kEmbMmaWarp) tmem_alloc(tmem_slot, TMEM_COLS);
  tc_fence_before();
  __syncthreads();
  tc_fence_after();
  const uint32_t tmem = *tmem_slot;

  if (warp == kEmbMmaWarp) {
    // ================================================================================================ MMA issuer
    if (elect_one()) {
      const uint32_t mid_bytes = (uint32_t)(D * ROWB), out_bytes = (uint32_t)(16 * ROWB);
      mbar_expect_tx(bar_w, n_mid * mid_bytes + out_bytes);
      for (int l = 0; l < n_mid; ++l) bulk_g2s(W + l * mid_bytes, a.wmid_img[l], mid_bytes, bar_w);
      bulk_g2s(W + n_mid * mid_bytes, a.wout_img, out_bytes, bar_w);
      mbar_wait(bar_w, 0);
      const uint32_t a_addr = smem_u32(A), w_addr = smem_u32(W);
      const uint32_t idesc_mid = make_idesc<kBf16>(D), idesc_out = make_idesc<kBf16>(16);
      int done[kEmbGroups], total[kEmbGroups], left = 0;
#pragma unroll
      for (int g = 0; g < kEmbGroups; ++g) {
        int t = 0;                                           // tiles of this CTA owned by warpgroup g
        for (long long it = g; blockIdx.x + it * gridDim.x < n_tiles; it += kEmbGroups) ++t;
        done[g] = 0; total[g] = t * H; left += total[g];
      }
      for (uint32_t spins = 0; left > 0; ++spins) {
        // whichever warpgroup has its operand ready gets its layer issued: job j of a group is layer j % H of its
        // tile j / H, and a_ready[g] completes once per job
#pragma unroll
        for (int g = 0; g < kEmbGroups; ++g) {
          if (done[g] < total[g] && mbar_test(&a_ready[g], done[g] & 1)) {
            tc_fence_after();
            const int l = done[g] % H;
            if (l < n_mid) issue_layer<kBf16, 128>(a_addr + g * TILE, w_addr + l * mid_bytes, ROWB, D, tmem + g * D, idesc_mid);
            else issue_layer<kBf16, 128>(a_addr + g * TILE, w_addr + n_mid * mid_bytes, ROWB, 16, tmem + g * D, idesc_out);
            umma_commit(&acc_full[g]);
            ++done[g]; --left; spins = 0;
          }
        }
        if ((spins & 0xfffffu) == 0xfffffu && mbar_stalled(spins)) __trap();                 // never hang the GPU: a lost arrival becomes an error
      }
    }
  } else {
    // ================================================================================================ compute groups
    const int g = warp >> 2, q = warp & 3;
    const uint32_t r = q * 32 + lane;                        // row of the tile = TMEM lane owned by this thread
    const uint32_t acc = tmem + ((uint32_t)(q * 32) << 16) + g * D;
    uint8_t* At = A + g * TILE;
    int job = 0;
    long long tile = blockIdx.x + (long long)g * gridDim.x;
    float4 f_next = make_float4(0.f, 0.f, 0.f, 0.f);
    if (tile < n_tiles && tile * kRows + r < a.n_rows) f_next = __ldg(a.feat + tile * kRows + r);
    for (; tile < n_tiles; tile += (long long)kEmbGroups * gridDim.x) {
      const long long row = tile * kRows + r;
      const float4 f = f_next;
      {                                                      // features of this warpgroup's next tile
        const long long nrow = row + (long long)kEmbGroups * gridDim.x * kRows;
        f_next = nrow < a.n_rows ? __ldg(a.feat + nrow) : make_float4(0.f, 0.f, 0.f, 0.f);
      }
      // ---- layer 0 (K = 3) on the FFMA pipe, pinned order (R3); relu -> bf16 -> operand tile
#pragma unroll
      for (int c0 = 0; c0 < D; c0 += 32) {
        uint32_t pk[16];
#pragma unroll
        for (int i = 0; i < 16; ++i) {
          float y[2];
#pragma unroll
          for (int h = 0; h < 2; ++h) {
            const int c = c0 + 2 * i + h;
            float s = __fmaf_rn(f.x, a.w0t[c], 0.0f);
            s = __fmaf_rn(f.y, a.w0t[D + c], s);
            s = __fmaf_rn(f.z, a.w0t[2 * D + c], s);
            y[h] = __fadd_rn(s, a.b0[c]);
          }
          pk[i] = pack_bf16x2_relu(y[0], y[1]);
        }
        store_row32(At, r, c0, pk);
      }
      fence_proxy_async();
      mbar_arrive(&a_ready[g]);
      // ---- D -> D tensor layers: relu(acc + b) -> bf16 -> the same tile, in place (the MMA has finished with it)
      for (int l = 0; l < n_mid; ++l, ++job) {
        mbar_wait(&acc_full[g], job & 1);
        tc_fence_after();
#pragma unroll
        for (int c0 = 0; c0 < D; c0 += 32) {
          uint32_t v[32], pk[16];
          tmem_ld32(acc + c0, v);
#pragma unroll
          for (int i = 0; i < 16; ++i)
            pk[i] = pack_bf16x2_relu(__fadd_rn(__uint_as_float(v[2 * i]), a.bmid[l][c0 + 2 * i]),
                                     __fadd_rn(__uint_as_float(v[2 * i + 1]), a.bmid[l][c0 + 2 * i + 1]));
          store_row32(At, r, c0, pk);
        }
        tc_fence_before();
        fence_proxy_async();
        mbar_arrive(&a_ready[g]);
      }
      // ---- output layer D -> 4 (N padded to 16): fp32, linear (R20)
      mbar_wait(&acc_full[g], job & 1);
      ++job;
      tc_fence_after();
      uint32_t v[4];
      tmem_ld4(acc, v);
      tc_fence_before();
      if (row < a.n_rows)
        a.emb[row] = make_float4(__fadd_rn(__uint_as_float(v[0]), a.bout[0]), __fadd_rn(__uint_as_float(v[1]), a.bout[1]),
                                 __fadd_rn(__uint_as_float(v[2]), a.bout[2]), __fadd_rn(__uint_as_float(v[3]), a.bout[3]));
    }
  }
  tc_fence_before();
  __syncthreads();
  if (warp == kEmbMmaWarp) tmem_dealloc(tmem, TMEM_COLS);
}

template <int D>
bool emb_ws_launch(etx_ctx* c, const EmbWsArgs& a, cudaStream_t s) {
  auto kern = embed_ws_kernel<D>;
  const int smem = emb_ws_smem<D>(a.n_mid) + 1024;
  if (smem > 227 * 1024) return false;
  opt_in_smem(c, kern, smem);
  const int tiles = (a.n_rows + kRows - 1) / kRows;
  const int grid = tiles < c->sm_count ? tiles : c->sm_count;     // one persistent CTA per SM
  if (grid <= 0) return true;
  kern<<<grid, kEmbThreads, smem, s>>>(a);
  c->launches++;
  return true;
}

}  // namespace

// bf16 mode with at most kEmbMaxMid + 1 hidden layers; returns false (nothing launched) when the shape is not
// covered, and the caller falls back to embed_umma_kernel
bool launch_embed_ws(etx_ctx* c, int n_hits, cudaStream_t s) {
  const int D = c->hp.emb_hidden, H = c->hp.emb_n_hidden_layers, n_mid = H - 1;
  if (c->precision != ETX_BF16 || n_mid < 0 || n_mid > kEmbMaxMid || (D != 64 && D != 128) || c->hp.emb_dim != 4) return false;
  EmbWsArgs a;
  const HostLayer& l0 = c->layers[c->i_emb0];
  for (int n = 0; n < D; ++n) {
    for (int k = 0; k < 3; ++k) a.w0t[k * D + n] = l0.W[(size_t)n * 3 + k];
    a.b0[n] = l0.b[n];
  }
  for (int l = 0; l < n_mid; ++l) {
    const HostLayer& lm = c->layers[c->i_emb0 + 1 + l];
    for (int n = 0; n < D; ++n) a.bmid[l][n] = lm.b[n];
    a.wmid_img[l] = lm.dev.Wtc;
  }
  const HostLayer& lo = c->layers[c->i_emb0 + H];
  for (int n = 0; n < 4; ++n) a.bout[n] = lo.b[n];
  a.wout_img = lo.dev.Wtc;
  a.feat = c->feat_emb; a.emb = c->emb; a.n_rows = n_hits; a.n_mid = n_mid;
  return D == 64 ? emb_ws_launch<64>(c, a, s) : emb_ws_launch<128>(c, a, s);
}

}  // namespace etx
