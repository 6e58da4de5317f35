// tc_common.cuh — sm_100a building blocks of the mixed-precision kernels: 5th-generation tensor cores
// (tcgen05.mma with shared-memory operands and TMEM accumulators), mbarriers, TMEM allocation / loads, and the
// error-compensated TF32 split ("3xTF32": x = hi + lo with hi, lo in TF32; a b ~ hi_a hi_b + lo_a hi_b + hi_a lo_b,
// fp32 accumulate), which brings a TF32 contraction to fp32-level accuracy.
// Internal; nothing here is shared with oracle/.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>
#include <string.h>

namespace tc {

// ---- shared-memory operand layout: K-major, 128-byte swizzle --------------------------------------------------
// A panel holds `rows` x 32 tf32 (one 128-byte row per matrix row); 8-row groups of 1024 bytes; inside a group the
// 16-byte chunk index is XORed with the row index (canonical SWIZZLE_128B).  Panels must be 1024-byte aligned.
__host__ __device__ __forceinline__ constexpr uint32_t sw128_offset(uint32_t row, uint32_t k /* 0..31 */) {
  return (row >> 3) * 1024u + (row & 7u) * 128u + ((((k >> 2) ^ (row & 7u)) & 7u) << 4) + ((k & 3u) << 2);
}

// UMMA shared-memory matrix descriptor (sm_100 format): start address >> 4 in bits [0,14), leading byte offset >> 4
// in [16,30) (unused for swizzled K-major operands), stride byte offset >> 4 in [32,46) = 1024 B between 8-row
// groups, version = 1 in [46,48), layout type SWIZZLE_128B = 2 in [61,64).
__device__ __forceinline__ uint64_t make_desc_sw128(uint32_t smem_addr) {
  uint64_t d = 0;
  d |= (uint64_t)((smem_addr & 0x3FFFFu) >> 4);
  d |= (uint64_t)1 << 16;
  d |= (uint64_t)(1024u >> 4) << 32;
  d |= (uint64_t)1 << 46;
  d |= (uint64_t)2 << 61;
  return d;
}

// Instruction descriptor for kind::tf32, fp32 accumulate, K-major A and B, M x N tile.
__host__ __device__ __forceinline__ constexpr uint32_t make_idesc_tf32(uint32_t M, uint32_t N) {
  return (1u << 4)          // c_format = F32
       | (2u << 7)          // a_format = TF32
       | (2u << 10)         // b_format = TF32
       | ((N >> 3) << 17)   // n_dim
       | ((M >> 4) << 24);  // m_dim
}

// Same layout for 16-bit operands (BF16): a panel row of 128 bytes holds 64 K-columns.
__host__ __device__ __forceinline__ constexpr uint32_t sw128_offset_b16(uint32_t row, uint32_t k /* 0..63 */) {
  return (row >> 3) * 1024u + (row & 7u) * 128u + ((((k >> 3) ^ (row & 7u)) & 7u) << 4) + ((k & 7u) << 1);
}

// Instruction descriptor for kind::f16 with BF16 operands, fp32 accumulate, K-major A and B, M x N tile (K = 16).
__host__ __device__ __forceinline__ constexpr uint32_t make_idesc_bf16(uint32_t M, uint32_t N) {
  return (1u << 4)          // c_format = F32
       | (1u << 7)          // a_format = BF16
       | (1u << 10)         // b_format = BF16
       | ((N >> 3) << 17)   // n_dim
       | ((M >> 4) << 24);  // m_dim
}

__device__ __forceinline__ uint32_t smem_u32(const void *p) { return (uint32_t)__cvta_generic_to_shared(p); }

// D[tmem] (+)= A[smem] B[smem], 16-bit operands (kind::f16; the instruction descriptor says BF16).
__device__ __forceinline__ void mma_f16_ss(uint32_t tmem_d, uint64_t desc_a, uint64_t desc_b, uint32_t idesc,
                                           uint32_t accumulate) {
  asm volatile(
      "{\n\t"
      ".reg .pred p;\n\t"
      "setp.ne.b32 p, %4, 0;\n\t"
      "tcgen05.mma.cta_group::1.kind::f16 [%0], %1, %2, %3, p;\n\t"
      "}\n" ::"r"(tmem_d), "l"(desc_a), "l"(desc_b), "r"(idesc), "r"(accumulate)
      : "memory");
}

// D[tmem] (+)= A[smem] B[smem]; issued by ONE thread on behalf of the CTA.
__device__ __forceinline__ void mma_tf32_ss(uint32_t tmem_d, uint64_t desc_a, uint64_t desc_b, uint32_t idesc,
                                            uint32_t accumulate) {
  asm volatile(
      "{\n\t"
      ".reg .pred p;\n\t"
      "setp.ne.b32 p, %4, 0;\n\t"
      "tcgen05.mma.cta_group::1.kind::tf32 [%0], %1, %2, %3, p;\n\t"
      "}\n" ::"r"(tmem_d), "l"(desc_a), "l"(desc_b), "r"(idesc), "r"(accumulate)
      : "memory");
}

// D[tmem] (+)= A[tmem] B[smem]: the A operand comes from tensor memory (lane = row, one 32-bit column per K element).
__device__ __forceinline__ void mma_tf32_ts(uint32_t tmem_d, uint32_t tmem_a, uint64_t desc_b, uint32_t idesc,
                                            uint32_t accumulate) {
  asm volatile(
      "{\n\t"
      ".reg .pred p;\n\t"
      "setp.ne.b32 p, %4, 0;\n\t"
      "tcgen05.mma.cta_group::1.kind::tf32 [%0], [%1], %2, %3, p;\n\t"
      "}\n" ::"r"(tmem_d), "r"(tmem_a), "l"(desc_b), "r"(idesc), "r"(accumulate)
      : "memory");
}

// tcgen05.st 32x32b.x32: lane l of the warp writes 32 consecutive columns of TMEM lane 32 (warp % 4) + l.
__device__ __forceinline__ void tmem_st32_nowait(uint32_t taddr, const uint32_t r[32]) {
  asm volatile("tcgen05.st.sync.aligned.32x32b.x32.b32 [%0], {%1, %2, %3, %4, %5, %6, %7, %8, %9, %10, %11, %12, %13, %14, %15, %16, %17, %18, %19, %20, %21, %22, %23, %24, %25, %26, %27, %28, %29, %30, %31, %32};\n" ::"r"(taddr), "r"(r[0]), "r"(r[1]), "r"(r[2]), "r"(r[3]), "r"(r[4]), "r"(r[5]), "r"(r[6]), "r"(r[7]), "r"(r[8]), "r"(r[9]), "r"(r[10]), "r"(r[11]), "r"(r[12]), "r"(r[13]), "r"(r[14]), "r"(r[15]), "r"(r[16]), "r"(r[17]), "r"(r[18]), "r"(r[19]), "r"(r[20]), "r"(r[21]), "r"(r[22]), "r"(r[23]), "r"(r[24]), "r"(r[25]), "r"(r[26]), "r"(r[27]), "r"(r[28]), "r"(r[29]), "r"(r[30]), "r"(r[31]) : "memory");
}
__device__ __forceinline__ void tmem_wait_st() { asm volatile("tcgen05.wait::st.sync.aligned;\n" ::: "memory"); }

// Arrive on an mbarrier when all tcgen05.mma issued so far by this thread have completed.
__device__ __forceinline__ void mma_commit(uint64_t *mbar) {
  asm volatile("tcgen05.commit.cta_group::1.mbarrier::arrive::one.shared::cluster.b64 [%0];\n" ::"r"(smem_u32(mbar))
               : "memory");
}

__device__ __forceinline__ void fence_before_sync() { asm volatile("tcgen05.fence::before_thread_sync;\n" ::: "memory"); }
__device__ __forceinline__ void fence_after_sync() { asm volatile("tcgen05.fence::after_thread_sync;\n" ::: "memory"); }
// generic-proxy writes to shared memory -> visible to the async proxy (tcgen05.mma operand reads)
__device__ __forceinline__ void fence_proxy_async() { asm volatile("fence.proxy.async.shared::cta;\n" ::: "memory"); }

__device__ __forceinline__ void mbar_init(uint64_t *mbar, uint32_t count) {
  asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;\n" ::"r"(smem_u32(mbar)), "r"(count) : "memory");
}
__device__ __forceinline__ void fence_mbar_init() { asm volatile("fence.mbarrier_init.release.cluster;\n" ::: "memory"); }

__device__ __forceinline__ void mbar_wait(uint64_t *mbar, uint32_t parity) {
  asm volatile(
      "{\n\t"
      ".reg .pred p;\n\t"
      "WAIT_%=:\n\t"
      "mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n\t"
      "@p bra DONE_%=;\n\t"
      "bra WAIT_%=;\n\t"
      "DONE_%=:\n\t"
      "}\n" ::"r"(smem_u32(mbar)), "r"(parity)
      : "memory");
}

__device__ __forceinline__ void mbar_arrive_expect_tx(uint64_t *mbar, uint32_t bytes) {
  asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;\n" ::"r"(smem_u32(mbar)), "r"(bytes) : "memory");
}

// 1-D bulk copy global -> shared (TMA engine, no tensor map), completion counted on an mbarrier.
__device__ __forceinline__ void bulk_g2s(void *smem_dst, const void *gsrc, uint32_t bytes, uint64_t *mbar) {
  asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];\n" ::"r"(
                   smem_u32(smem_dst)),
               "l"(gsrc), "r"(bytes), "r"(smem_u32(mbar))
               : "memory");
}

// named barrier for a subset of the CTA's warps
__device__ __forceinline__ void bar_sync(int id, int nthreads) {
  asm volatile("bar.sync %0, %1;\n" ::"r"(id), "r"(nthreads) : "memory");
}

// ---- TMEM ---------------------------------------------------------------------------------------------------
// One warp allocates `cols` (power of two >= 32) columns and writes the base address to shared memory.
template <int COLS>
__device__ __forceinline__ void tmem_alloc(uint32_t *dst_in_smem) {
  asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], %1;\n" ::"r"(smem_u32(dst_in_smem)),
               "n"(COLS)
               : "memory");
  asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;\n" ::: "memory");
}
template <int COLS>
__device__ __forceinline__ void tmem_dealloc(uint32_t base) {
  asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, %1;\n" ::"r"(base), "n"(COLS) : "memory");
}

// tcgen05.ld 32x32b: lane l of the warp reads TMEM lane (32 * (warp % 4) + l), 8 consecutive 32-bit columns.
__device__ __forceinline__ void tmem_ld8(uint32_t taddr, float v[8]) {
  uint32_t r[8];
  asm volatile("tcgen05.ld.sync.aligned.32x32b.x8.b32 {%0, %1, %2, %3, %4, %5, %6, %7}, [%8];\n"
               : "=r"(r[0]), "=r"(r[1]), "=r"(r[2]), "=r"(r[3]), "=r"(r[4]), "=r"(r[5]), "=r"(r[6]), "=r"(r[7])
               : "r"(taddr)
               : "memory");
  asm volatile("tcgen05.wait::ld.sync.aligned;\n" ::: "memory");
#pragma unroll
  for (int i = 0; i < 8; ++i) v[i] = __uint_as_float(r[i]);
}
// two independent x8 loads in flight, one wait
__device__ __forceinline__ void tmem_ld8x2(uint32_t ta, uint32_t tb, float a[8], float b[8]) {
  uint32_t r[8], s[8];
  asm volatile("tcgen05.ld.sync.aligned.32x32b.x8.b32 {%0, %1, %2, %3, %4, %5, %6, %7}, [%8];\n"
               : "=r"(r[0]), "=r"(r[1]), "=r"(r[2]), "=r"(r[3]), "=r"(r[4]), "=r"(r[5]), "=r"(r[6]), "=r"(r[7])
               : "r"(ta)
               : "memory");
  asm volatile("tcgen05.ld.sync.aligned.32x32b.x8.b32 {%0, %1, %2, %3, %4, %5, %6, %7}, [%8];\n"
               : "=r"(s[0]), "=r"(s[1]), "=r"(s[2]), "=r"(s[3]), "=r"(s[4]), "=r"(s[5]), "=r"(s[6]), "=r"(s[7])
               : "r"(tb)
               : "memory");
  asm volatile("tcgen05.wait::ld.sync.aligned;\n" ::: "memory");
#pragma unroll
  for (int i = 0; i < 8; ++i) { a[i] = __uint_as_float(r[i]); b[i] = __uint_as_float(s[i]); }
}

// 16 consecutive columns of this thread's TMEM lane; no wait (pair with tmem_wait_ld before using r[])
__device__ __forceinline__ void tmem_ld16_nowait(uint32_t taddr, uint32_t r[16]) {
  asm volatile("tcgen05.ld.sync.aligned.32x32b.x16.b32 {%0, %1, %2, %3, %4, %5, %6, %7, %8, %9, %10, %11, %12, %13, %14, %15}, [%16];\n"
               : "=r"(r[0]), "=r"(r[1]), "=r"(r[2]), "=r"(r[3]), "=r"(r[4]), "=r"(r[5]), "=r"(r[6]), "=r"(r[7]), "=r"(r[8]), "=r"(r[9]), "=r"(r[10]), "=r"(r[11]), "=r"(r[12]), "=r"(r[13]), "=r"(r[14]), "=r"(r[15])
               : "r"(taddr)
               : "memory");
}
// 32 consecutive columns of this thread's TMEM lane; no wait (pair with tmem_wait_ld before using r[])
__device__ __forceinline__ void tmem_ld32_nowait(uint32_t taddr, uint32_t r[32]) {
  asm volatile("tcgen05.ld.sync.aligned.32x32b.x32.b32 {%0, %1, %2, %3, %4, %5, %6, %7, %8, %9, %10, %11, %12, %13, %14, %15, %16, %17, %18, %19, %20, %21, %22, %23, %24, %25, %26, %27, %28, %29, %30, %31}, [%32];\n"
               : "=r"(r[0]), "=r"(r[1]), "=r"(r[2]), "=r"(r[3]), "=r"(r[4]), "=r"(r[5]), "=r"(r[6]), "=r"(r[7]), "=r"(r[8]), "=r"(r[9]), "=r"(r[10]), "=r"(r[11]), "=r"(r[12]), "=r"(r[13]), "=r"(r[14]), "=r"(r[15]), "=r"(r[16]), "=r"(r[17]), "=r"(r[18]), "=r"(r[19]), "=r"(r[20]), "=r"(r[21]), "=r"(r[22]), "=r"(r[23]), "=r"(r[24]), "=r"(r[25]), "=r"(r[26]), "=r"(r[27]), "=r"(r[28]), "=r"(r[29]), "=r"(r[30]), "=r"(r[31])
               : "r"(taddr)
               : "memory");
}
__device__ __forceinline__ void tmem_ld8_nowait(uint32_t taddr, uint32_t r[8]) {
  asm volatile("tcgen05.ld.sync.aligned.32x32b.x8.b32 {%0, %1, %2, %3, %4, %5, %6, %7}, [%8];\n"
               : "=r"(r[0]), "=r"(r[1]), "=r"(r[2]), "=r"(r[3]), "=r"(r[4]), "=r"(r[5]), "=r"(r[6]), "=r"(r[7])
               : "r"(taddr)
               : "memory");
}
__device__ __forceinline__ void tmem_wait_ld() { asm volatile("tcgen05.wait::ld.sync.aligned;\n" ::: "memory"); }
// NC columns (multiple of 8) starting at taddr into r[], issued as x32 / x16 / x8 pieces, no wait
template <int NC>
__device__ __forceinline__ void tmem_ld_cols_nowait(uint32_t taddr, uint32_t *r) {
  static_assert(NC % 8 == 0 && NC <= 64, "");
  if constexpr (NC >= 32) {
    tmem_ld32_nowait(taddr, r);
    tmem_ld_cols_nowait<NC - 32>(taddr + 32, r + 32);
  } else if constexpr (NC >= 16) {
    tmem_ld16_nowait(taddr, r);
    tmem_ld_cols_nowait<NC - 16>(taddr + 16, r + 16);
  } else if constexpr (NC == 8) {
    tmem_ld8_nowait(taddr, r);
  }
}

// ---- numerics -------------------------------------------------------------------------------------------------
// x = hi + lo, both representable in TF32 (10 explicit mantissa bits): hi = rna(x), lo = rna(x - hi).
__device__ __forceinline__ void split_tf32(float x, float &hi, float &lo) {
  uint32_t h, l;
  asm("cvt.rna.tf32.f32 %0, %1;" : "=r"(h) : "f"(x));
  hi = __uint_as_float(h);
  const float rem = x - hi;
  asm("cvt.rna.tf32.f32 %0, %1;" : "=r"(l) : "f"(rem));
  lo = __uint_as_float(l);
}

// x = p0 + p1 + p2 with every piece representable in BF16 (8 significant bits each, 24 together: all of fp32's):
// p0 = rn(x), p1 = rn(x - p0), p2 = rn(x - p0 - p1); returned as the 16-bit patterns.
__device__ __forceinline__ uint32_t bf16_bits_rn(float x) {
  uint32_t u = __float_as_uint(x);
  u += 0x7fffu + ((u >> 16) & 1u);                          // round to nearest even (finite inputs)
  return u >> 16;
}
__device__ __forceinline__ void split_bf16x3(float x, uint32_t &p0, uint32_t &p1, uint32_t &p2) {
  p0 = bf16_bits_rn(x);
  const float r1 = x - __uint_as_float(p0 << 16);
  p1 = bf16_bits_rn(r1);
  const float r2 = r1 - __uint_as_float(p1 << 16);
  p2 = bf16_bits_rn(r2);
}

// fp32 tanh and its derivative from u = exp(-2|x|) in (0, 1] (ex2.approx) and r = 1 / (1 + u) (rcp.approx):
//   tanh x = sign(x) (1 - u) r,    1 - tanh^2 x = 4 u r^2.
// The derivative is formed without the cancellation of 1 - t^2, so it keeps fp32 relative accuracy in the saturated
// regime (|x| large), where most of the fitting net's units sit with random weights.  2 MUFU + 5..7 FMA-pipe ops.
__device__ __forceinline__ void tanh_d_f32(float x, float &t, float &dt) {
  float u, r;
  const float a = fabsf(x) * -2.885390081777927f;   // -2 log2(e) |x|
  asm("ex2.approx.ftz.f32 %0, %1;" : "=f"(u) : "f"(a));
  const float d = u + 1.0f;
  asm("rcp.approx.ftz.f32 %0, %1;" : "=f"(r) : "f"(d));
  t = copysignf((1.0f - u) * r, x);
  const float ur = u * r;
  dt = 4.0f * ur * r;
}
__device__ __forceinline__ float tanh_f32(float x) {
  float u, r;
  const float a = fabsf(x) * -2.885390081777927f;
  asm("ex2.approx.ftz.f32 %0, %1;" : "=f"(u) : "f"(a));
  const float d = u + 1.0f;
  asm("rcp.approx.ftz.f32 %0, %1;" : "=f"(r) : "f"(d));
  return copysignf((1.0f - u) * r, x);
}

// tanh of an argument that is already scaled by 2 log2(e): 1 - 2 / (2^a + 1).  ex2, add, rcp, fma.
__device__ __forceinline__ float tanh_prescaled_f32(float a) {
  float e, r;
  asm("ex2.approx.ftz.f32 %0, %1;" : "=f"(e) : "f"(a));
  const float d = e + 1.0f;
  asm("rcp.approx.ftz.f32 %0, %1;" : "=f"(r) : "f"(d));
  return fmaf(-2.0f, r, 1.0f);
}
#define TC_2LOG2E 2.885390081777927f

// packed fp32 FMA (FFMA2): (d.x, d.y) = (a.x b.x + c.x, a.y b.y + c.y)
__device__ __forceinline__ float2 ffma2(float2 a, float2 b, float2 c) {
  unsigned long long ua, ub, uc, ud;
  asm("mov.b64 %0, {%1, %2};" : "=l"(ua) : "f"(a.x), "f"(a.y));
  asm("mov.b64 %0, {%1, %2};" : "=l"(ub) : "f"(b.x), "f"(b.y));
  asm("mov.b64 %0, {%1, %2};" : "=l"(uc) : "f"(c.x), "f"(c.y));
  asm("fma.rn.f32x2 %0, %1, %2, %3;" : "=l"(ud) : "l"(ua), "l"(ub), "l"(uc));
  float2 d;
  asm("mov.b64 {%0, %1}, %2;" : "=f"(d.x), "=f"(d.y) : "l"(ud));
  return d;
}

}  // namespace tc

// host-side BF16 rounding (round to nearest even), returned as the 16-bit pattern
static inline uint16_t tc_host_bf16_bits(float x) {
  uint32_t u;
  memcpy(&u, &x, 4);
  u += 0x7fffu + ((u >> 16) & 1u);
  return (uint16_t)(u >> 16);
}
static inline float tc_host_bf16_value(uint16_t b) {
  const uint32_t u = (uint32_t)b << 16;
  float y;
  memcpy(&y, &u, 4);
  return y;
}

// host-side TF32 rounding (round to nearest, ties away from zero: what cvt.rna.tf32.f32 does)
static inline float tc_host_tf32(float x) {
  uint32_t u;
  memcpy(&u, &x, 4);
  if ((u & 0x7f800000u) == 0x7f800000u) return x;
  u += 0x1000u;
  u &= 0xffffe000u;
  float y;
  memcpy(&y, &u, 4);
  return y;
}
