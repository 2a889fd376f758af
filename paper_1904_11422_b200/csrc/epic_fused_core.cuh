// Device code shared by the fused kernels (epic_fused.cu: support within 32 x 32; epic_wide.cu: support
// within 64 x 64): the 32-point ramped transform, the voltage prefetch / unpack, the gather of the
// 32 x 32 kernels, the product/accumulate column tasks and the ordered fix-up of split units.
// See the header comment of epic_fused.cu for the algorithm.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

#include "epic_internal.h"
#include "epic_packed.cuh"

namespace epic {
namespace {

constexpr int S = 32;        // support block side (cells)
constexpr int HS = 34;       // row stride of a shared plane in float4 cells (bank-conflict-free)
constexpr int PLANE = S * HS;  // float4 cells per pair-plane
constexpr int F = 4;         // pairs per batch
constexpr int MAXW = 2;      // prefetched word pairs per thread
constexpr int CHUNK = 2;     // fold: elements whose loads may be in flight together

constexpr int bitrev4(int v) { return ((v & 1) << 3) | ((v & 2) << 1) | ((v & 4) >> 1) | ((v & 8) >> 3); }

// fold: z[bitrev(y)] = in[y] + c in[y+16], y = 0..15, c = r^16.  `in` strides by `stride` float4
// cells; elements y + 16 with y >= NB are structurally zero and are not read.
template <int NB, int Y>
__device__ __forceinline__ void fold(C2 (&z)[16], const float4* __restrict__ in, int stride, float cr, float ci) {
  if constexpr (Y < 16) {
    const float4 a = in[Y * stride];
    float2 sr = make_float2(a.x, a.y), si = make_float2(a.z, a.w);
    if constexpr (Y < NB) {
      const float4 b = in[(Y + 16) * stride];
      const float2 br = make_float2(b.x, b.y), bi = make_float2(b.z, b.w);
      sr = __ffma2_rn(br, f2(cr), sr); sr = __ffma2_rn(neg2(bi), f2(ci), sr);
      si = __ffma2_rn(bi, f2(cr), si); si = __ffma2_rn(br, f2(ci), si);
    }
    z[bitrev4(Y)].re = sr; z[bitrev4(Y)].im = si;
    // bar.warp.sync is the one fence ptxas will not move shared loads across: without it all
    // loads are hoisted to the top of the task and the accumulators spill (128-register budget)
    if constexpr ((Y & (CHUNK - 1)) == CHUNK - 1 && Y < 15) __syncwarp();
    fold<NB, Y + 1>(z, in, stride, cr, ci);
  }
}

// One whole transform: `tw` points at the residue's TwSet words in shared memory.
template <int NB>
__device__ __forceinline__ void transform32(C2 (&z)[16], const float4* __restrict__ in, int stride,
                                            const float4* __restrict__ tw) {
  const float4 t0 = tw[0];
  fold<NB, 0>(z, in, stride, t0.x, t0.y);
  fft16_ramped(z, tw, t0.z, t0.w);
}

// ---------------------------------------------------------------- kernel parameters
struct FusedParams {
  const uint8_t* volt;       // [T][C][NPOL][A] 4+4-bit samples
  float* out;                // [C][planes][N][N]
  const uint2* cell_info;    // [32*32] cell slots sorted by entry count: x = (first entry << 8) | count,
                             // y = cell offset cy*HS + cx in a plane (0xFFFFFFFF: unused slot)
  int cell_stride;           // 32*32 when every channel has its own table (reading Q15), else 0
  const uint16_t* ent_ant;   // gather entries, sorted by block cell
  const float2* ent_tap;
  const float4* tw;          // [2Q][TWV]: the TwSet of every residue rho
  float* partial;            // scratch [grid][2 slots][NACC][16][NT]: partial sums of split units
  int native;                // input order [T][C][A][Np] instead of [T][C][Np][A]
  const float4* phasor;      // delay phasors, pair-packed [C][A], or nullptr
  int n_t, n_chan, n_ant, n_pol, n_planes;  // n_ant: antennas rounded up to a multiple of 4 (strides of E, prefetch slots)
  int n_ant_true;            // antennas of a voltage row
  int unaligned;             // n_ant_true % 4 != 0: voltage rows are not word-aligned, the tail group is short
  int n_ent;                 // gather entries (one layout)
  int R, Cc;                 // occupied rows / columns of the block
  int pairs_per_batch;       // pairs per batch the launch was sized for (epic_fused_kernel's FF)
  int nb;                    // batches per unit
  long long total;           // n_chan * Q * nb batches in all
};

// Per-thread voltage slots, fixed for the kernel's lifetime: slot k covers antennas a..a+3 of pair j
// of every batch (j < 0: unused).  Voltage rows are read as aligned 32-bit words.
struct PrefetchSlots {
  int j[MAXW], a[MAXW];
};

template <int NT, int FF = F>
__device__ __forceinline__ void prefetch_init(const FusedParams& P, int tid, PrefetchSlots& ps) {
  const int ag = P.n_ant >> 2;
#pragma unroll
  for (int k = 0; k < MAXW; ++k) {
    const int i = tid + k * NT;
    ps.j[k] = -1; ps.a[k] = 0;
    if (i < FF * ag) { ps.j[k] = i / ag; ps.a[k] = (i - ps.j[k] * ag) << 2; }
  }
}

// global -> registers: the voltages of batch b of channel c (F pairs x A antennas).  Time samples
// past n_t read as the zero sample.
// Antenna counts that are no multiple of 4: voltage rows are not word-aligned, so the four samples of a slot
// (antennas a0 .. a0+3 of time samples t_lo / t_hi of channel c) are fetched as bytes; antennas past the end read
// as the zero sample.  Returns (word of the lo plane, word of the hi plane) as prefetch_batch makes them.
__device__ __noinline__ uint2 fetch_slot_bytes(const uint8_t* __restrict__ volt, int n_t, int n_chan, int n_ant, int n_pol,
                                               int native, int c, int t_lo, int t_hi, int a0) {
  const size_t row_bytes = (size_t)n_pol * n_ant;
  uint32_t wlo = 0u, whi = 0u;
  for (int i = 0; i < 4; ++i) {
    if (a0 + i >= n_ant) break;
    if (native && n_pol == 2) {
      if (t_lo < n_t) {
        const uint8_t* src = volt + ((size_t)t_lo * n_chan + c) * row_bytes + 2 * (a0 + i);
        wlo |= (uint32_t)__ldg(src) << (8 * i);
        whi |= (uint32_t)__ldg(src + 1) << (8 * i);
      }
    } else {
      const uint8_t* base = volt + (size_t)c * row_bytes + a0 + i;
      if (t_lo < n_t) wlo |= (uint32_t)__ldg(base + (size_t)t_lo * n_chan * row_bytes) << (8 * i);
      if (t_hi < n_t) whi |= (uint32_t)__ldg(base + (size_t)t_hi * n_chan * row_bytes + (n_pol == 2 ? n_ant : 0)) << (8 * i);
    }
  }
  return make_uint2(wlo, whi);
}

template <int NT, int FF = F>
__device__ __forceinline__ void prefetch_batch(const FusedParams& P, const PrefetchSlots& ps, int c, int b,
                                               uint32_t (&wlo)[MAXW], uint32_t (&whi)[MAXW]) {
  const int tmul = P.n_pol == 2 ? 1 : 2, thi = P.n_pol == 2 ? 0 : 1, hi_off = P.n_pol == 2 ? P.n_ant_true : 0;
  const size_t row_bytes = (size_t)P.n_pol * P.n_ant_true;
#pragma unroll
  for (int k = 0; k < MAXW; ++k) {
    wlo[k] = 0u; whi[k] = 0u;
    if (ps.j[k] >= 0) {
      const int t_lo = (b * FF + ps.j[k]) * tmul, t_hi = t_lo + thi;
      if (P.unaligned) {  // rare path, kept out of line: inlined it cost the 128-register kernels 88 bytes of spills
        const uint2 w = fetch_slot_bytes(P.volt, P.n_t, P.n_chan, P.n_ant_true, P.n_pol, P.native, c, t_lo, t_hi, ps.a[k]);
        wlo[k] = w.x; whi[k] = w.y;
        continue;
      }
      if (P.native && P.n_pol == 2) {  // (a X, a Y) byte pairs: two words hold this slot's four antennas
        if (t_lo < P.n_t) {
          const uint32_t* src = reinterpret_cast<const uint32_t*>(
              P.volt + ((size_t)t_lo * P.n_chan + c) * row_bytes + 2 * ps.a[k]);
          deinterleave_pols(__ldg(src), __ldg(src + 1), wlo[k], whi[k]);
        }
        continue;
      }
      const uint8_t* base = P.volt + (size_t)c * row_bytes + ps.a[k];
      if (t_lo < P.n_t) wlo[k] = __ldg(reinterpret_cast<const uint32_t*>(base + (size_t)t_lo * P.n_chan * row_bytes));
      if (t_hi < P.n_t) whi[k] = __ldg(reinterpret_cast<const uint32_t*>(base + (size_t)t_hi * P.n_chan * row_bytes + hi_off));
    }
  }
}

// registers -> E[F][A] (float4 per antenna), S1.  EB: E holds one 32-bit word per antenna instead, the four
// values as bytes biased by 8 (epic_packed.cuh), for the integer gather of the delta kernels.
template <bool EB = false>
__device__ __forceinline__ void unpack_batch(const FusedParams& P, const PrefetchSlots& ps, float4* __restrict__ E,
                                             const uint32_t (&wlo)[MAXW], const uint32_t (&whi)[MAXW], int c) {
  if constexpr (EB) {
    uint32_t* Eb = reinterpret_cast<uint32_t*>(E);
#pragma unroll
    for (int k = 0; k < MAXW; ++k)
      if (ps.j[k] >= 0) *reinterpret_cast<uint4*>(Eb + ps.j[k] * P.n_ant + ps.a[k]) = unpack_words_b8(wlo[k], whi[k]);
    return;
  }
#pragma unroll
  for (int k = 0; k < MAXW; ++k)
    if (ps.j[k] >= 0)
      unpack_words(wlo[k], whi[k], E + ps.j[k] * P.n_ant + ps.a[k], (int)(threadIdx.x >> 1),
                   P.phasor ? P.phasor + (size_t)c * P.n_ant_true + ps.a[k] : nullptr);
}

// S3 for the batch: every thread owns the cell slots tid + j*NT of the plan's list and sums their
// gather lists, in table order, for all F pair-planes (collisions sum).  The
// list holds every cell of the R x 32 block (empty ones are written as zeros) sorted by entry
// count, so the 32 cells of a warp have (nearly) equal trip counts.
// EB (delta kernel, at most 16 antennas per cell, no delay phasors): the four values of an antenna
// are bytes 0..15 of one word, so a cell's sum is ONE integer add per antenna and pair -- the byte
// sums stay below 256 -- turned into floats once per cell: exact, like the float adds it replaces.
template <int NT, bool DELTA, bool STG = false, bool EB = false, int FF = F>
__device__ __forceinline__ void gather_batch(const FusedParams& P, const float4* __restrict__ E,
                                             float4* __restrict__ gh, const uint2 (&info)[S * S / NT],
                                             const uint16_t* __restrict__ ant_s = nullptr,
                                             const float2* __restrict__ tap_s = nullptr) {
#pragma unroll
  for (int j = 0; j < S * S / NT; ++j) {
    if (info[j].y == 0xFFFFFFFFu) continue;
    const uint32_t beg = info[j].x >> 8, cnt = info[j].x & 0xFFu;
    if constexpr (EB) {
      const uint32_t* Eb = reinterpret_cast<const uint32_t*>(E);
      uint32_t sum[FF];
#pragma unroll
      for (int f = 0; f < FF; ++f) sum[f] = 0u;
      for (uint32_t e = beg; e < beg + cnt; ++e) {
        const uint32_t* ea = Eb + __ldg(P.ent_ant + e);
#pragma unroll
        for (int f = 0; f < FF; ++f) sum[f] += ea[f * P.n_ant];
      }
      const float2 bias = f2(-(12582912.0f + 8.0f * (float)cnt));  // mantissa trick of epic_packed.cuh, cnt biases of 8
      float4* dst = gh + info[j].y;
#pragma unroll
      for (int f = 0; f < FF; ++f) {
        const float2 vr = __fadd2_rn(make_float2(biased_byte_to_float_bits(sum[f], 0), biased_byte_to_float_bits(sum[f], 1)), bias);
        const float2 vi = __fadd2_rn(make_float2(biased_byte_to_float_bits(sum[f], 2), biased_byte_to_float_bits(sum[f], 3)), bias);
        dst[f * PLANE] = make_float4(vr.x, vr.y, vi.x, vi.y);
      }
      continue;
    }
    float2 sr[FF], si[FF];
#pragma unroll
    for (int f = 0; f < FF; ++f) { sr[f] = make_float2(0.0f, 0.0f); si[f] = make_float2(0.0f, 0.0f); }
    for (uint32_t e = beg; e < beg + cnt; ++e) {
      const float4* ea = E + (STG ? (uint32_t)ant_s[e] : (uint32_t)__ldg(P.ent_ant + e));
      if (DELTA) {
#pragma unroll
        for (int f = 0; f < FF; ++f) {
          const float4 v = ea[f * P.n_ant];
          sr[f] = __fadd2_rn(sr[f], make_float2(v.x, v.y));
          si[f] = __fadd2_rn(si[f], make_float2(v.z, v.w));
        }
      } else {
        const float2 w = STG ? tap_s[e] : __ldg(P.ent_tap + e);
        const float2 wr = f2(w.x), wi = f2(w.y);
#pragma unroll
        for (int f = 0; f < FF; ++f) {
          const float4 v = ea[f * P.n_ant];
          const float2 vr = make_float2(v.x, v.y), vi = make_float2(v.z, v.w);
          sr[f] = __ffma2_rn(vr, wr, sr[f]); sr[f] = __ffma2_rn(neg2(vi), wi, sr[f]);
          si[f] = __ffma2_rn(vi, wr, si[f]); si[f] = __ffma2_rn(vr, wi, si[f]);
        }
      }
    }
    float4* dst = gh + info[j].y;
#pragma unroll
    for (int f = 0; f < FF; ++f) dst[f * PLANE] = make_float4(sr[f].x, sr[f].y, si[f].x, si[f].y);
  }
}

// ---------------------------------------------------------------- the two transform roles
// rows: thread = (pair f, row y, h); 32 cells of the row -> outputs l1 = 2k + h, in place.
// The caller guarantees both h-threads of a row sit in one warp and separates loads from stores
// with __syncwarp().
template <int NB>
__device__ __forceinline__ void row_task(float4* __restrict__ row, const float4* __restrict__ tw, int h, bool valid) {
  C2 z[16];
  transform32<NB>(z, row, 1, tw);
  __syncwarp();
  if (valid) {
#pragma unroll
    for (int k = 0; k < 16; ++k) row[2 * k + h] = make_float4(z[k].re.x, z[k].re.y, z[k].im.x, z[k].im.y);
  }
}

// columns + S5 + S6: thread = (l1, rho); outputs m = 2Q k + rho, k = 0..15.
// acc[k] = (|A_lo|^2, |A_hi|^2) sums in registers (one or two products).
template <int NB>
__device__ __forceinline__ void col_task(const float4* __restrict__ col, const float4* __restrict__ tw,
                                         float2 (&acc)[16]) {
  C2 z[16];
  transform32<NB>(z, col, HS, tw);
#pragma unroll
  for (int k = 0; k < 16; ++k) {
    acc[k] = __ffma2_rn(z[k].re, z[k].re, acc[k]);
    acc[k] = __ffma2_rn(z[k].im, z[k].im, acc[k]);
  }
}

// out_accum planes of one pixel += v (reading Q14: {XX} | {XX,YY} | {XX,YY,Re XY,Im XY,Re YX,Im YX})
template <int NPROD>
__device__ __forceinline__ void add_pixel(float* __restrict__ px, size_t plane, const float* v) {
  px[0] += v[0];
  if constexpr (NPROD >= 2) px[plane] += v[1];
  if constexpr (NPROD == 4) {  // YX = conj(XY)
    px[2 * plane] += v[2];
    px[3 * plane] += v[3];
    px[4 * plane] += v[2];
    px[5 * plane] -= v[3];
  }
}

// Adds the parked partial sums of every unit whose time range was split between CTAs, in CTA
// order.  One CTA per unit, same thread <-> pixel mapping as the main kernel.
template <int Q, int NPROD, bool TC = false>
__global__ void __launch_bounds__(64 * Q) epic_fused_fixup(FusedParams P, int main_grid) {
  // NT threads with KPT pixels each, as in the main kernel (the tensor-core kernel: its 256 epilogue threads)
  constexpr int NT = 64 * Q, KPT = 16, N = 32 * Q, NACC = NPROD == 4 ? 4 : (NPROD == 2 ? 2 : 1);
  const int unit = blockIdx.x, tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  const long long G = main_grid, first = (long long)unit * P.nb, last = first + P.nb - 1;
  const int b_lo = (int)(((first + 1) * G - 1) / P.total), b_hi = (int)(((last + 1) * G - 1) / P.total);
  if (b_lo == b_hi) return;  // the unit ran in one CTA and was added directly
  const int l1 = (warp & 1) * 16 + (lane >> 1);
  const int rho = (warp >> 1) * 2 + (lane & 1);
  const int c = unit / Q, l2 = unit - c * Q;
  const size_t plane = (size_t)N * N;
  float* o = P.out + (size_t)c * P.n_planes * plane + (Q * l1 + l2) + (size_t)rho * N;
  size_t kstride = (size_t)2 * Q * N;
  if constexpr (TC) {  // tensor-core kernel: thread = (image row m, 16 columns l1), see epic_tc_kernel
    o = P.out + (size_t)c * P.n_planes * plane + (size_t)((warp & 3) * 32 + lane) * N + Q * KPT * (warp >> 2) + l2;
    kstride = Q;
  }
  for (int k = 0; k < KPT; ++k) {
    float v[NACC];
#pragma unroll
    for (int q = 0; q < NACC; ++q) v[q] = 0.0f;
    for (int b = b_lo; b <= b_hi; ++b) {
      const int slot = (first <= P.total * b / G) ? 0 : 1;  // does the segment start the CTA's range?
      const float* part = P.partial + ((size_t)(b * 2 + slot) * NACC * KPT) * NT + tid;
#pragma unroll
      for (int q = 0; q < NACC; ++q) v[q] += part[(size_t)(q * KPT + k) * NT];
    }
    add_pixel<NPROD>(o + k * kstride, plane, v);
  }
}

// Four-product variant: the 64 accumulators of a thread (16 pixels x {XX, YY, Re XY, Im XY}) do not fit
// beside the 64 data registers at two CTAs per SM, so they are parked in tensor memory (TMEM) and
// updated 4 pixels at a time: load 16 words, 16 FMAs, store 16 words.  Layout: column 4 k + {0,1,2,3};
// XY = A_lo conj(A_hi) (reading Q11).
template <int NB>
__device__ __forceinline__ void col_task_tmem(const float4* __restrict__ col, const float4* __restrict__ tw,
                                              uint32_t taddr) {
  C2 z[16];
  uint32_t r[2][16];
  tmem_ld16_issue(taddr, r[0]);  // the first 4 pixels' accumulators travel during the transform
  transform32<NB>(z, col, HS, tw);
#pragma unroll
  for (int c = 0; c < 4; ++c) {
    tmem_wait_ld();
    if (c < 3) tmem_ld16_issue(taddr + 16 * (c + 1), r[(c + 1) & 1]);  // next 4 pixels, during this update
    float a[16];
#pragma unroll
    for (int i = 0; i < 16; ++i) a[i] = __uint_as_float(r[c & 1][i]);
#pragma unroll
    for (int kk = 0; kk < 4; ++kk) {
      const C2& v = z[4 * c + kk];
      float2 p = make_float2(a[4 * kk], a[4 * kk + 1]);
      p = __ffma2_rn(v.re, v.re, p);
      p = __ffma2_rn(v.im, v.im, p);
      a[4 * kk] = p.x; a[4 * kk + 1] = p.y;
      a[4 * kk + 2] = fmaf(v.re.x, v.re.y, a[4 * kk + 2]); a[4 * kk + 2] = fmaf(v.im.x, v.im.y, a[4 * kk + 2]);
      a[4 * kk + 3] = fmaf(v.im.x, v.re.y, a[4 * kk + 3]); a[4 * kk + 3] = fmaf(-v.re.x, v.im.y, a[4 * kk + 3]);
    }
    tmem_st16(taddr + 16 * c, a);
  }
  tmem_wait_st();
}

}  // namespace
}  // namespace epic
