// PTX wrappers, UMMA descriptors and operand conversions shared by the tcgen05 kernels (k_mlp_umma.cu,
// k_mlp_ws.cu).  Internal to the CUDA library; nothing here is shared with oracle/.
#pragma once

#include "etx_internal.h"

namespace etx {
namespace umma {

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
// A wait is declared lost only by wall-clock time (about 20 s), never by a poll count: under a debugger, a sanitizer,
// time-slicing or a throttled clock a healthy wait can take any number of polls.  Called every 2^20 polls.
static __device__ __noinline__ bool mbar_stalled(uint32_t spins) {
  unsigned long long now;
  asm volatile("mov.u64 %0, %%globaltimer;" : "=l"(now));
  __shared__ unsigned long long first_seen;              // any waiter's first slow-path time stamp of this CTA
  if (spins == 0xfffffu) { first_seen = now; return false; }
  // another waiter may have stored a LATER first_seen between this thread's clock read and this load: the unsigned
  // difference would wrap and read as a stall, so a time stamp that is not in the past never counts
  const unsigned long long t0 = first_seen;
  return now > t0 && now - t0 > 20000000000ull;
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
    if (!done && (spins & 0xfffffu) == 0xfffffu && mbar_stalled(spins)) __trap();   // never hang the GPU: a lost arrival becomes an error
  }
}
// one lane of the (converged) warp.  ptxas knows a region guarded by elect.sync runs single-threaded, so the
// operands of the tcgen05 instructions inside it move to uniform registers without a per-instruction
// ELECT / R2UR.BROADCAST loop (which `lane == 0` costs: ~75 cycles per MMA instead of a few)
__device__ __forceinline__ bool elect_one() {
  uint32_t p;
  asm volatile("{\n\t.reg .pred p;\n\telect.sync _|p, 0xffffffff;\n\tselp.u32 %0, 1, 0, p;\n\t}" : "=r"(p));
  return p != 0;
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

__device__ __forceinline__ void mbar_arrive(uint64_t* bar) {
  asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(smem_u32(bar)) : "memory");
}
__device__ __forceinline__ bool mbar_test(uint64_t* bar, uint32_t parity) {      // non-blocking
  uint32_t done;
  asm volatile(
      "{\n\t.reg .pred p;\n\t"
      "mbarrier.test_wait.parity.shared::cta.b64 p, [%1], %2;\n\t"
      "selp.u32 %0, 1, 0, p;\n\t}"
      : "=r"(done) : "r"(smem_u32(bar)), "r"(parity) : "memory");
  return done != 0;
}
// two fp32 -> bf16x2 (RNE), lo in the low half; the .relu form clamps negative inputs to +0 first, which for a
// monotone rounding is the same as rounding relu(x) (R3, R20)
__device__ __forceinline__ uint32_t pack_bf16x2_relu(float lo, float hi) {
  uint32_t r;
  asm("cvt.rn.relu.bf16x2.f32 %0, %1, %2;" : "=r"(r) : "f"(hi), "f"(lo));
  return r;
}

// 32 lanes x 32 columns without the wait (so that two loads can be in flight)
__device__ __forceinline__ void tmem_ld32_nowait(uint32_t taddr, uint32_t (&v)[32]) {
  asm volatile(
      "tcgen05.ld.sync.aligned.32x32b.x32.b32 "
      "{%0, %1, %2, %3, %4, %5, %6, %7, %8, %9, %10, %11, %12, %13, %14, %15, "
      "%16, %17, %18, %19, %20, %21, %22, %23, %24, %25, %26, %27, %28, %29, %30, %31}, [%32];"
      : "=r"(v[0]), "=r"(v[1]), "=r"(v[2]), "=r"(v[3]), "=r"(v[4]), "=r"(v[5]), "=r"(v[6]), "=r"(v[7]),
        "=r"(v[8]), "=r"(v[9]), "=r"(v[10]), "=r"(v[11]), "=r"(v[12]), "=r"(v[13]), "=r"(v[14]), "=r"(v[15]),
        "=r"(v[16]), "=r"(v[17]), "=r"(v[18]), "=r"(v[19]), "=r"(v[20]), "=r"(v[21]), "=r"(v[22]), "=r"(v[23]),
        "=r"(v[24]), "=r"(v[25]), "=r"(v[26]), "=r"(v[27]), "=r"(v[28]), "=r"(v[29]), "=r"(v[30]), "=r"(v[31])
      : "r"(taddr) : "memory");
}
__device__ __forceinline__ void tmem_ld_wait() { asm volatile("tcgen05.wait::ld.sync.aligned;" ::: "memory"); }

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
// R21: q = clamp(rne(x * (1 / s_x)), +-127).  Returned in the LOW BYTE of the result (two's complement), the
// upper bytes are not meaningful: pack_i8x4 takes low bytes only.  Clamping to the integer bounds first and then
// adding 1.5 * 2^23 rounds to nearest-even in the fp32 adder and leaves the integer in the low mantissa bits --
// the same value as rintf -> clamp -> cvt for every finite input, with four full-rate instructions instead of the
// quarter-rate FRND and F2I (which bounded the INT8 kernels: ~65 k conversions per 128-edge tile).
__device__ __forceinline__ int quant_i8(float x, float inv_s) {
  float r = __fmul_rn(x, inv_s);
  r = fminf(fmaxf(r, -127.0f), 127.0f);
  return (int)__float_as_uint(__fadd_rn(r, 12582912.0f));
}
__device__ __forceinline__ uint32_t pack_i8x4(int a, int b, int c, int d) {     // low bytes of a, b, c, d
  const uint32_t lo = __byte_perm((uint32_t)a, (uint32_t)b, 0x0040), hi = __byte_perm((uint32_t)c, (uint32_t)d, 0x0040);
  return __byte_perm(lo, hi, 0x5410);
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

}  // namespace umma
}  // namespace etx
