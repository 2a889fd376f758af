// Device helpers shared by the packed (f32x2) kernels: epic_fused.cu and epic_tiled.cu.
//
// Every complex value is carried as a PAIR of planes in the two halves of f32x2 registers
// (sm_100 FFMA2/FADD2: one issue slot, two FP32 lanes; the twiddle is one broadcast .F32 operand):
// (lo, hi) = (pol X, pol Y) of one time sample when n_pol == 2, or two consecutive time samples
// when n_pol == 1.  A shared/global memory cell is a float4 (re_lo, re_hi, im_lo, im_hi).
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

namespace epic {
namespace {

constexpr int TWV = 5;       // float4 words of twiddles per residue (TwSet)

// ---------------------------------------------------------------- packed complex pair
struct C2 { float2 re, im; };  // (lo, hi) halves = two independent planes

__device__ __forceinline__ float2 f2(float v) { return make_float2(v, v); }  // FFMA2 takes it as one .F32 operand
__device__ __forceinline__ float2 neg2(float2 v) { return make_float2(-v.x, -v.y); }

// The transform one thread computes (rows and columns alike):
//
//   X[k] = sum_{y<32} in[y] r^y W_16^{y k},  k = 0..15,   r = W_N^{rho}  (|r| = 1)
//        = sum_{y<16} (in[y] + r^16 in[y+16]) r^y W_16^{y k}
//
// The residue ramp r^y is absorbed into the butterflies: decimation in time gives, for a length-n
// sub-transform T_n(s, r_n),  T_n[k], T_n[k + n/2] = T_{n/2}(s_even, r_n^2)[k] +- (r_n W_n^k) T_{n/2}(s_odd, r_n^2)[k],
// so level n = 2, 4, 8, 16 uses the twiddles r^{16/n} W_n^k: nine complex numbers per residue
// (W_n^{k + n/4} = i W_n^k is a register swap), computed in double on the host.
struct TwSet {
  float cr, ci;              // r^16        (fold)
  float w2r, w2i;            // r^8         (level 2)
  float w4r, w4i;            // r^4         (level 4, k = 0; k = 1 is i times it)
  float w8r[2], w8i[2];      // r^2 W_8^k   (level 8, k = 0, 1)
  float w16r[4], w16i[4];    // r W_16^k    (level 16, k = 0..3)
};

// shared-memory image of a TwSet: TWV float4 words
//   [0] = (cr, ci, w2r, w2i)  [1] = (w4r, w4i, w8r0, w8i0)  [2] = (w8r1, w8i1, w16r0, w16i0)
//   [3] = (w16r1, w16i1, w16r2, w16i2)  [4] = (w16r3, w16i3, 0, 0)

// radix-2 DIT butterfly on packed pairs: (a, b) <- (a + w b, a - w b); 6 FFMA2
__device__ __forceinline__ void bfly(C2& a, C2& b, float wr, float wi) {
  C2 p;
  p.re = __ffma2_rn(b.re, f2(wr), a.re); p.re = __ffma2_rn(neg2(b.im), f2(wi), p.re);
  p.im = __ffma2_rn(b.im, f2(wr), a.im); p.im = __ffma2_rn(b.re, f2(wi), p.im);
  b.re = __ffma2_rn(a.re, f2(2.0f), neg2(p.re));
  b.im = __ffma2_rn(a.im, f2(2.0f), neg2(p.im));
  a = p;
}
// the same with twiddle i w = (-wi, wr)
__device__ __forceinline__ void bfly_i(C2& a, C2& b, float wr, float wi) { bfly(a, b, -wi, wr); }

// z holds s[y] = in[y] + r^16 in[y+16] in bit-reversed order; on return z[k] = X[k].
// Twiddles are read from the residue's shared-memory TwSet level by level (short live ranges).
__device__ __forceinline__ void fft16_ramped(C2 (&z)[16], const float4* __restrict__ tw, float w2r, float w2i) {
#pragma unroll
  for (int b = 0; b < 16; b += 2) bfly(z[b], z[b + 1], w2r, w2i);
  const float4 t1 = tw[1];
#pragma unroll
  for (int b = 0; b < 16; b += 4) { bfly(z[b], z[b + 2], t1.x, t1.y); bfly_i(z[b + 1], z[b + 3], t1.x, t1.y); }
  const float4 t2 = tw[2];
#pragma unroll
  for (int b = 0; b < 16; b += 8) {
    bfly(z[b], z[b + 4], t1.z, t1.w);   bfly(z[b + 1], z[b + 5], t2.x, t2.y);
    bfly_i(z[b + 2], z[b + 6], t1.z, t1.w); bfly_i(z[b + 3], z[b + 7], t2.x, t2.y);
  }
  const float4 t3 = tw[3], t4 = tw[4];
  bfly(z[0], z[8], t2.z, t2.w);    bfly(z[1], z[9], t3.x, t3.y);
  bfly(z[2], z[10], t3.z, t3.w);   bfly(z[3], z[11], t4.x, t4.y);
  bfly_i(z[4], z[12], t2.z, t2.w); bfly_i(z[5], z[13], t3.x, t3.y);
  bfly_i(z[6], z[14], t3.z, t3.w); bfly_i(z[7], z[15], t4.x, t4.y);
}

// 8-point version: z holds the input in 3-bit bit-reversed order; twiddles (base q):
// q^4 (level 2), q^2 (level 4; k = 1 is i times it), q W_8^k, k = 0, 1 (level 8).
__device__ __forceinline__ void fft8_ramped(C2 (&z)[8], float w2r, float w2i, float w4r, float w4i,
                                            float w80r, float w80i, float w81r, float w81i) {
#pragma unroll
  for (int b = 0; b < 8; b += 2) bfly(z[b], z[b + 1], w2r, w2i);
#pragma unroll
  for (int b = 0; b < 8; b += 4) { bfly(z[b], z[b + 2], w4r, w4i); bfly_i(z[b + 1], z[b + 3], w4r, w4i); }
  bfly(z[0], z[4], w80r, w80i);   bfly(z[1], z[5], w81r, w81i);
  bfly_i(z[2], z[6], w80r, w80i); bfly_i(z[3], z[7], w81r, w81i);
}

// S1 (reading Q1).  Four samples per 32-bit word: high nibbles are the real
// parts, low nibbles the imaginary parts, two's complement.  n ^ 8 = sext4(n) + 8 in 0..15;
// dropping that byte into the mantissa of 12582912.0f (0x4B400000) and subtracting 12582920.0f
// gives sext4(n) exactly, with no integer-to-float conversion instruction.
__device__ __forceinline__ float biased_byte_to_float_bits(uint32_t w, int i) {
  return __uint_as_float(__byte_perm(w, 0x4B400000u, 0x7650u + (uint32_t)i));
}

// word pair (lo plane, hi plane) of antennas a0..a0+3 -> E[a0..a0+3] = (re_lo, re_hi, im_lo, im_hi).
// `ph` (or nullptr): the four antennas' delay phasors, pair-packed the same way; each sample is
// multiplied by its phasor (PAPER.md:122 delay compensation; reading Q19).
__device__ __forceinline__ void unpack_words(uint32_t wlo, uint32_t whi, float4* __restrict__ e, int rot,
                                             const float4* __restrict__ ph = nullptr) {
  const uint32_t rl = ((wlo >> 4) & 0x0F0F0F0Fu) ^ 0x08080808u, il = (wlo & 0x0F0F0F0Fu) ^ 0x08080808u;
  const uint32_t rh = ((whi >> 4) & 0x0F0F0F0Fu) ^ 0x08080808u, ih = (whi & 0x0F0F0F0Fu) ^ 0x08080808u;
  const float2 bias = f2(-12582920.0f);
#pragma unroll
  for (int k = 0; k < 4; ++k) {
    // lanes store their four cells in rotated order so that a quarter-warp covers all 8 bank groups
    const int i = (k + rot) & 3;
    float2 re = __fadd2_rn(make_float2(biased_byte_to_float_bits(rl, i), biased_byte_to_float_bits(rh, i)), bias);
    float2 im = __fadd2_rn(make_float2(biased_byte_to_float_bits(il, i), biased_byte_to_float_bits(ih, i)), bias);
    if (ph) {
      const float4 p = __ldg(ph + i);
      const float2 pr = make_float2(p.x, p.y), pi = make_float2(p.z, p.w);
      const float2 r2 = __ffma2_rn(re, pr, neg2(__fmul2_rn(im, pi)));
      im = __ffma2_rn(re, pi, __fmul2_rn(im, pr));
      re = r2;
    }
    e[i] = make_float4(re.x, re.y, im.x, im.y);
  }
}

// The untransposed input order [T][C][A][Np] with two polarisations: 8 consecutive
// bytes hold (a0 X, a0 Y, a1 X, a1 Y | a2 X, a2 Y, a3 X, a3 Y); split them into the X and Y words.
__device__ __forceinline__ void deinterleave_pols(uint32_t w0, uint32_t w1, uint32_t& wlo, uint32_t& whi) {
  wlo = __byte_perm(w0, w1, 0x6420u);
  whi = __byte_perm(w0, w1, 0x7531u);
}

// Compact form of the same unpack for large antenna counts: one 32-bit word per antenna holding
// the four biased nibbles as bytes (re_lo+8, re_hi+8, im_lo+8, im_hi+8); converted at use.
__device__ __forceinline__ uint4 unpack_words_b8(uint32_t wlo, uint32_t whi) {
  const uint32_t rl = ((wlo >> 4) & 0x0F0F0F0Fu) ^ 0x08080808u, il = (wlo & 0x0F0F0F0Fu) ^ 0x08080808u;
  const uint32_t rh = ((whi >> 4) & 0x0F0F0F0Fu) ^ 0x08080808u, ih = (whi & 0x0F0F0F0Fu) ^ 0x08080808u;
  uint32_t o[4];
#pragma unroll
  for (int i = 0; i < 4; ++i) {
    const uint32_t re = __byte_perm(rl, rh, 0x0040u + 0x11u * (uint32_t)i);  // bytes (rl_i, rh_i, -, -)
    const uint32_t im = __byte_perm(il, ih, 0x0040u + 0x11u * (uint32_t)i);
    o[i] = __byte_perm(re, im, 0x5410u);
  }
  return make_uint4(o[0], o[1], o[2], o[3]);
}
__device__ __forceinline__ void b8_to_pair(uint32_t w, float2& vr, float2& vi) {
  const float2 bias = f2(-12582920.0f);
  vr = __fadd2_rn(make_float2(biased_byte_to_float_bits(w, 0), biased_byte_to_float_bits(w, 1)), bias);
  vi = __fadd2_rn(make_float2(biased_byte_to_float_bits(w, 2), biased_byte_to_float_bits(w, 3)), bias);
}

// ---------------------------------------------------------------- TMEM as per-thread accumulator storage
// Blackwell tensor memory (256 KB/SM, 128 lanes x 512 columns of 32 bits) is used here without
// the tensor cores: a warp owns the 32 lanes of its quadrant (warp % 4), and tcgen05.ld/st with
// shape 32x32b.x16 move 16 consecutive columns of a thread's own lane to/from 16 registers.
// Measured on B200 (round 1 probe): a load+add+store round trip sustains 360 B/clk/SM each way.
// asynchronous: the registers are valid only after tmem_wait_ld()
__device__ __forceinline__ void tmem_ld16_issue(uint32_t taddr, uint32_t (&r)[16]) {
  asm volatile(
      "tcgen05.ld.sync.aligned.32x32b.x16.b32 {%0,%1,%2,%3,%4,%5,%6,%7,%8,%9,%10,%11,%12,%13,%14,%15}, [%16];\n"
      : "=r"(r[0]), "=r"(r[1]), "=r"(r[2]), "=r"(r[3]), "=r"(r[4]), "=r"(r[5]), "=r"(r[6]), "=r"(r[7]), "=r"(r[8]),
        "=r"(r[9]), "=r"(r[10]), "=r"(r[11]), "=r"(r[12]), "=r"(r[13]), "=r"(r[14]), "=r"(r[15])
      : "r"(taddr));
}
__device__ __forceinline__ void tmem_ld8_issue(uint32_t taddr, uint32_t (&r)[8]) {
  asm volatile("tcgen05.ld.sync.aligned.32x32b.x8.b32 {%0,%1,%2,%3,%4,%5,%6,%7}, [%8];\n"
               : "=r"(r[0]), "=r"(r[1]), "=r"(r[2]), "=r"(r[3]), "=r"(r[4]), "=r"(r[5]), "=r"(r[6]), "=r"(r[7])
               : "r"(taddr));
}
__device__ __forceinline__ void tmem_wait_ld() { asm volatile("tcgen05.wait::ld.sync.aligned;\n" ::: "memory"); }
__device__ __forceinline__ void tmem_ld16(uint32_t taddr, float (&v)[16]) {
  uint32_t r[16];
  tmem_ld16_issue(taddr, r);
  tmem_wait_ld();
#pragma unroll
  for (int i = 0; i < 16; ++i) v[i] = __uint_as_float(r[i]);
}
__device__ __forceinline__ void tmem_st16(uint32_t taddr, const float (&v)[16]) {
  asm volatile(
      "tcgen05.st.sync.aligned.32x32b.x16.b32 [%0], {%1,%2,%3,%4,%5,%6,%7,%8,%9,%10,%11,%12,%13,%14,%15,%16};\n" ::"r"(taddr),
      "r"(__float_as_uint(v[0])), "r"(__float_as_uint(v[1])), "r"(__float_as_uint(v[2])), "r"(__float_as_uint(v[3])),
      "r"(__float_as_uint(v[4])), "r"(__float_as_uint(v[5])), "r"(__float_as_uint(v[6])), "r"(__float_as_uint(v[7])),
      "r"(__float_as_uint(v[8])), "r"(__float_as_uint(v[9])), "r"(__float_as_uint(v[10])), "r"(__float_as_uint(v[11])),
      "r"(__float_as_uint(v[12])), "r"(__float_as_uint(v[13])), "r"(__float_as_uint(v[14])), "r"(__float_as_uint(v[15]))
      : "memory");
}
__device__ __forceinline__ void tmem_wait_st() { asm volatile("tcgen05.wait::st.sync.aligned;\n" ::: "memory"); }

// One warp allocates NCOLS columns for the CTA (result through shared memory) / frees them.
template <int NCOLS>
__device__ __forceinline__ uint32_t tmem_alloc_cta(uint32_t* slot_smem, int warp) {
  if (warp == 0) {
    const uint32_t sa = (uint32_t)__cvta_generic_to_shared(slot_smem);
    asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], %1;\n" ::"r"(sa), "n"(NCOLS) : "memory");
    asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;\n" ::: "memory");
  }
  asm volatile("tcgen05.fence::before_thread_sync;\n" ::: "memory");
  __syncthreads();
  asm volatile("tcgen05.fence::after_thread_sync;\n" ::: "memory");
  return *slot_smem;
}
template <int NCOLS>
__device__ __forceinline__ void tmem_free_cta(uint32_t tbase, int warp) {
  asm volatile("tcgen05.fence::before_thread_sync;\n" ::: "memory");
  __syncthreads();
  if (warp == 0) asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, %1;\n" ::"r"(tbase), "n"(NCOLS) : "memory");
}

// ---------------------------------------------------------------- tcgen05.mma (5th-generation tensor cores)
// Shared-memory operand descriptor, K-major, no swizzle: the operand is a grid of 8-row x 16-byte
// core matrices (128 contiguous bytes each); `sbo` = byte distance between core matrices adjacent
// along M/N (groups of 8 rows), `lbo` = between the two 8-element K chunks of one K = 16 step.
// Bits: [0,14) address >> 4, [16,30) lbo >> 4, [32,46) sbo >> 4, [46,48) version = 1 (sm_100),
// [61,64) layout type 0.  Checked against a host GEMM by a probe before use.
__device__ __forceinline__ uint64_t umma_desc(uint32_t smem_addr, uint32_t lbo, uint32_t sbo) {
  return (uint64_t)((smem_addr & 0x3FFFFu) >> 4) | ((uint64_t)((lbo >> 4) & 0x3FFFu) << 16) |
         ((uint64_t)((sbo >> 4) & 0x3FFFu) << 32) | ((uint64_t)1 << 46);
}
// Instruction descriptor of kind::f16 with BF16 operands, FP32 accumulator, both operands K-major:
// bits [4,6) D format (1 = f32), [7,10) A format (1 = bf16), [10,13) B format, 13 negate A,
// [17,23) N >> 3, [24,29) M >> 4.
__host__ __device__ constexpr uint32_t umma_idesc_bf16(int M, int N, bool negate_a) {
  return (1u << 4) | (1u << 7) | (1u << 10) | ((negate_a ? 1u : 0u) << 13) | ((uint32_t)(N >> 3) << 17) |
         ((uint32_t)(M >> 4) << 24);
}
// D[tmem] (+)= A[smem] * B[smem]^T, issued by ONE thread for the CTA; asynchronous.
__device__ __forceinline__ void umma_bf16(uint32_t d_tmem, uint64_t desc_a, uint64_t desc_b, uint32_t idesc,
                                          uint32_t accumulate) {
  asm volatile(
      "{\n\t.reg .pred p;\n\tsetp.ne.b32 p, %4, 0;\n\t"
      "tcgen05.mma.cta_group::1.kind::f16 [%0], %1, %2, %3, p;\n\t}\n" ::"r"(d_tmem),
      "l"(desc_a), "l"(desc_b), "r"(idesc), "r"(accumulate)
      : "memory");
}
// The mbarrier receives one arrival when every MMA issued so far by this thread has completed.
__device__ __forceinline__ void umma_commit(uint64_t* bar) {
  asm volatile("tcgen05.commit.cta_group::1.mbarrier::arrive::one.shared::cluster.b64 [%0];\n" ::"r"(
                   (uint32_t)__cvta_generic_to_shared(bar))
               : "memory");
}
__device__ __forceinline__ void mbar_init(uint64_t* bar, uint32_t count) {
  asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;\n" ::"r"((uint32_t)__cvta_generic_to_shared(bar)), "r"(count)
               : "memory");
}
// Waits for the phase with the given parity; traps instead of hanging if it never completes.
__device__ __forceinline__ void mbar_wait(uint64_t* bar, uint32_t parity) {
  const uint32_t a = (uint32_t)__cvta_generic_to_shared(bar);
  uint32_t done = 0;
  for (int spin = 0; spin < (1 << 26) && !done; ++spin)
    asm volatile(
        "{\n\t.reg .pred p;\n\tmbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n\tselp.b32 %0, 1, 0, p;\n\t}\n"
        : "=r"(done)
        : "r"(a), "r"(parity)
        : "memory");
  if (!done) __trap();
}
// generic-proxy shared-memory writes -> visible to the async proxy (tensor-core operand reads)
__device__ __forceinline__ void fence_smem_to_async_proxy() { asm volatile("fence.proxy.async.shared::cta;\n" ::: "memory"); }
__device__ __forceinline__ void tc_fence_before_sync() { asm volatile("tcgen05.fence::before_thread_sync;\n" ::: "memory"); }
__device__ __forceinline__ void tc_fence_after_sync() { asm volatile("tcgen05.fence::after_thread_sync;\n" ::: "memory"); }

}  // namespace
}  // namespace epic
