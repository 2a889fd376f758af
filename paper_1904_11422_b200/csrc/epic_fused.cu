// Fused EPIC path: unpack -> grid -> 2-D transform -> products -> accumulate in ONE kernel; the
// aperture/image planes never leave the SM (BASELINE.json north_star (1)-(4)).
//
// Applies when the occupied cells of the aperture fit a 32 x 32 box (after the circular
// relocation of epic_plan.cu; reading Q7) and N = 32*Q, Q in {2,4}.  With the support
// S = 32 cells a side the N x N image splits into Q*Q independent 32 x 32 sub-images
//
//   A[Q m1 + m2][Q l1 + l2] = sum_{y,x<32} G[y][x] W_N^{x l2} W_N^{y m2} W_32^{x l1 + y m1},
//
// so the structurally-zero rows/columns of the padded plane are never transformed (a pruned
// decimation-in-frequency 2-D FFT whose first log2 Q stages per axis are phase ramps).
//
// Packing.  Every complex value is carried as a PAIR of planes in the two halves of f32x2
// registers (sm_100 FFMA2/FADD2/FMUL2: one issue slot, two FP32 lanes): (lo, hi) = (pol X, pol Y)
// of one time sample when n_pol == 2, or two consecutive time samples when n_pol == 1.  Both
// halves see the same twiddles, so the whole transform is packed arithmetic; a shared-memory
// cell is a float4 (re_lo, re_hi, im_lo, im_hi).
//
// Work unit = (channel c, column residue l2); its CTA owns the image columns l = Q l1 + l2 and
// keeps their accumulators in registers for the unit's whole time range.  One 32-point transform
// with residue rho is split over two threads h = 0,1 (outputs m1 = 2k + h):
//
//   X[2Q k + rho'] = sum_{y<16} (in[y] + r^16 in[y+16]) r^y W_16^{y k},  rho' = rho + Q h,  r = W_N^{rho'}
//
// i.e. a fold and a 16-point radix-2 FFT whose twiddles carry the ramp r^y (nine per-residue
// complex numbers read from shared memory; see TwSet).  Rows (along x, rho = l2) and columns
// (along y, rho = m2) run the SAME code, so the hot loop is a few KB of instructions shared by
// all warps.  (The first version of this kernel unrolled every residue with immediate twiddles:
// 109 KB of code, instruction-fetch bound at 0.36 of the roofline; profiles/r01_fused_c2_ncu.md.)
//
//   per batch of F pairs (F time samples when n_pol == 2):
//     prefetch  next batch's 4+4-bit voltages, global -> registers (consumed one batch later)
//     gather    S3: every thread owns fixed cells of the R x 32 block and sums its (antenna, tap)
//               list in table order from the unpacked voltages E (no atomics, deterministic)
//     rows      S4 along x, thread = (pair, row y, h), in place
//     unpack    S1: the prefetched words -> E (float4 per antenna) for the NEXT batch
//     columns   S4 along y + S5 + S6: thread = (l1, rho'); 16 outputs -> products -> += registers
//   at the end of the unit's time range: one add per pixel into out_accum (directly, or through
//   the partial-sum fix-up kernel when the unit's time range was split between two CTAs).
#include <algorithm>
#include <cmath>
#include <cstdlib>
#include <cstring>
#include <type_traits>
#include <vector>

#include <cuda_bf16.h>

#include "epic_internal.h"
#include "epic_packed.cuh"
#include "epic_fused_core.cuh"

#include <mutex>

// Scratch of epic_image_noalloc (include/epic.h): the partial sums of split work units of the residue-group kernel,
// in a file-scope static device array instead of the plan's cudaMalloc'ed buffer.  80 MiB: 2 slots x (residues x
// products = 8) x 16 pixels x 256 threads x 4 B = 256 KiB per resident CTA, x 296 CTAs = 74 MiB on a 148-SM B200.  Every GPU that loads
// the library holds it until the process exits.  In HOST code this name is a host-side stand-in, not a device
// address: the address the kernels get comes from cudaGetSymbolAddress (noalloc_scratch_ptr below).
constexpr size_t EPIC_NOALLOC_SCRATCH_BYTES = (size_t)80 << 20;
static __device__ __align__(256) unsigned char epic_noalloc_scratch[EPIC_NOALLOC_SCRATCH_BYTES];

namespace epic {
namespace {

// PC: every channel has its own cell table (per-channel plans); a separate instantiation, because
// making the cell records loop-variant costs the one-layout kernels 1-2 % (measured).
// STG: the gather's (antenna, tap) tables are copied to shared memory once per CTA (tap kernels of
// one-layout plans whose tables fit beside two resident CTAs): their reads leave the L1/L2 path,
// C3 +2.8 % (measured); the delta kernels, whose table is 2 bytes per antenna, gain nothing.
// FF: pairs per batch
template <int Q, int NPROD, bool DELTA, int NB, bool PC, bool STG, int FF = F>
__global__ void __launch_bounds__(64 * Q, 2)
epic_fused_kernel(FusedParams P) {
  static_assert(!(STG && (DELTA || PC)), "staged tables: tap kernels of one-layout plans only");
  constexpr int NT = 64 * Q, N = 32 * Q, NACC = NPROD == 4 ? 4 : (NPROD == 2 ? 2 : 1);
  extern __shared__ __align__(16) unsigned char smem_raw[];
  float4* gh = reinterpret_cast<float4*>(smem_raw);  // [FF][32][HS]
  float4* tws = gh + FF * PLANE;                      // [2Q][TWV]
  float4* E = tws + 2 * Q * TWV;                     // [FF][A]
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;

  // static, contiguous share of the (unit-major, batch-minor) work list
  const long long g0 = P.total * (long long)blockIdx.x / gridDim.x;
  const long long g1 = P.total * (long long)(blockIdx.x + 1) / gridDim.x;
  if (g0 >= g1) return;
  constexpr bool TMEM = NPROD == 4;        // accumulators in tensor memory
  constexpr int TCOLS = Q == 4 ? 128 : 64;  // 64 columns per warp; warps w and w + 4 share a lane quadrant

  int unit = (int)(g0 / P.nb);
  uint2 info[S * S / NT];  // this thread's cells of the current channel's layout
#pragma unroll
  for (int j = 0; j < S * S / NT; ++j)
    info[j] = __ldg(P.cell_info + (PC ? (size_t)(unit / Q) * (S * S) : (size_t)0) + tid + j * NT);
  for (int i = tid; i < FF * PLANE; i += NT) gh[i] = make_float4(0.0f, 0.0f, 0.0f, 0.0f);  // rows >= R stay zero
  for (int i = tid; i < 2 * Q * TWV; i += NT) tws[i] = __ldg(P.tw + i);
  float2* tap_s = reinterpret_cast<float2*>(E + FF * P.n_ant);       // [n_ent] (STG only)
  uint16_t* ant_s = reinterpret_cast<uint16_t*>(tap_s + P.n_ent);   // [n_ent]
  if constexpr (STG) {
    for (int i = tid; i < P.n_ent; i += NT) { tap_s[i] = __ldg(P.ent_tap + i); ant_s[i] = __ldg(P.ent_ant + i); }
  }
  __syncthreads();

  // column role: 16 consecutive l1 x 2 residues per warp, the two residues of a column in ADJACENT
  // lanes: LDS.128 merges same-address lane pairs, so a warp's load of a row is 2 wavefronts for
  // 256 unique bytes (measured; lanes i and i+8 sharing an address do not merge: 4 wavefronts)
  const int l1 = (warp & 1) * 16 + (lane >> 1);
  const int rho = (warp >> 1) * 2 + (lane & 1);

  float2 acc[TMEM ? 1 : 16];
#pragma unroll
  for (int k = 0; k < (TMEM ? 1 : 16); ++k) acc[k] = make_float2(0.0f, 0.0f);
  __shared__ uint32_t tmem_slot;
  uint32_t tbase = 0u, taddr = 0u;
  if constexpr (TMEM) {
    tbase = tmem_alloc_cta<TCOLS>(&tmem_slot, warp);
    taddr = tbase + (((uint32_t)(warp & 3) * 32u) << 16) + (uint32_t)(warp >> 2) * 64u;
    float zero[16];
#pragma unroll
    for (int i = 0; i < 16; ++i) zero[i] = 0.0f;
#pragma unroll
    for (int c = 0; c < 4; ++c) tmem_st16(taddr + 16 * c, zero);
    tmem_wait_st();
  }

  // S6.  A unit whose whole time range ran in this CTA is added to out_accum directly (this CTA
  // is the only writer of those pixels).  When the equal split of the work list cut a unit's time
  // range between CTAs, each CTA parks its partial sums in the scratch (slot 0: the segment that
  // starts the CTA's range, slot 1: the one that ends it) and epic_fused_fixup adds them in CTA
  // order: no atomics anywhere, and the result does not depend on scheduling.
  auto flush = [&](int unit, bool complete, int slot) {
    const int c = unit / Q, l2 = unit - c * Q;
    const size_t plane = (size_t)N * N;
    float* o = P.out + (size_t)c * P.n_planes * plane + (Q * l1 + l2);
    float* part = P.partial + ((size_t)(blockIdx.x * 2 + slot) * NACC * 16) * NT + tid;
    if constexpr (TMEM) {
#pragma unroll
      for (int c = 0; c < 4; ++c) {
        float a[16], zero[16];
        tmem_ld16(taddr + 16 * c, a);
#pragma unroll
        for (int i = 0; i < 16; ++i) zero[i] = 0.0f;
        tmem_st16(taddr + 16 * c, zero);
#pragma unroll
        for (int kk = 0; kk < 4; ++kk) {
          const int k = 4 * c + kk;
          const float v[4] = {a[4 * kk], a[4 * kk + 1], a[4 * kk + 2], a[4 * kk + 3]};
          if (complete) {
            add_pixel<4>(o + (size_t)(2 * Q * k + rho) * N, plane, v);
          } else {
#pragma unroll
            for (int q = 0; q < 4; ++q) part[(size_t)(q * 16 + k) * NT] = v[q];
          }
        }
      }
      tmem_wait_st();
      return;
    }
#pragma unroll
    for (int k = 0; k < (TMEM ? 1 : 16); ++k) {
      float v[NACC];
      if constexpr (NPROD == 1) {
        v[0] = acc[k].x + acc[k].y;
      } else {
        v[0] = acc[k].x; v[1] = acc[k].y;
      }
      acc[k] = make_float2(0.0f, 0.0f);
      if (complete) {
        add_pixel<NPROD>(o + (size_t)(2 * Q * k + rho) * N, plane, v);
      } else {
#pragma unroll
        for (int q = 0; q < NACC; ++q) part[(size_t)(q * 16 + k) * NT] = v[q];
      }
    }
  };

  int b = (int)(g0 - (long long)unit * P.nb);
  const int first_unit = unit;
  int seg_begin = b;  // first batch of the current unit done by this CTA
  PrefetchSlots ps;
  prefetch_init<NT, FF>(P, tid, ps);
  uint32_t wlo[MAXW], whi[MAXW];
  prefetch_batch<NT, FF>(P, ps, unit / Q, b, wlo, whi);
  unpack_batch<DELTA>(P, ps, E, wlo, whi, unit / Q);
  __syncthreads();

  const int ntask = FF * P.R * 2;
  for (long long g = g0; g < g1; ++g) {
    int unit_n = unit, b_n = b + 1;
    if (b_n == P.nb) { b_n = 0; ++unit_n; }
    const bool more = g + 1 < g1;
    if (more) prefetch_batch<NT, FF>(P, ps, unit_n / Q, b_n, wlo, whi);

    gather_batch<NT, DELTA, STG, DELTA, FF>(P, E, gh, info, ant_s, tap_s);
    __syncthreads();

    const int l2 = unit % Q;
    for (int base = warp * 32; base < ntask; base += NT) {
      const int task = base + lane;
      const bool valid = task < ntask;
      // idle lanes transform the all-zero row 31 of plane 0 (never written: they exist only when R < 32)
      int f = 0, y = S - 1, h = 0;
      if (valid) { h = task & 1; const int p = task >> 1; f = p / P.R; y = p - f * P.R; }
      row_task<NB>(gh + f * PLANE + y * HS, tws + (l2 + Q * h) * TWV, h, valid);
    }
    __syncthreads();

    if (more) unpack_batch<DELTA>(P, ps, E, wlo, whi, unit_n / Q);  // E was last read by this batch's gather
#pragma unroll 1
    for (int f = 0; f < FF; ++f) {
      // launder the table offset: the twiddles are re-read per task, not held in 18 registers
      int tw_off = rho * TWV;
      asm volatile("" : "+r"(tw_off));
      if constexpr (TMEM) col_task_tmem<NB>(gh + f * PLANE + l1, tws + tw_off, taddr);
      else col_task<NB>(gh + f * PLANE + l1, tws + tw_off, acc);
    }

    if (unit_n != unit || !more) {
      flush(unit, seg_begin == 0 && b == P.nb - 1, unit == first_unit ? 0 : 1);
      seg_begin = 0;
    }
    if constexpr (PC) {
      if (unit_n / Q != unit / Q && more) {  // the next channel's cells (gather_batch is done with these)
#pragma unroll
        for (int j = 0; j < S * S / NT; ++j)
          info[j] = __ldg(P.cell_info + (size_t)(unit_n / Q) * (S * S) + tid + j * NT);
      }
    }
    unit = unit_n; b = b_n;
    __syncthreads();  // next batch's E is complete; gh is free
  }
  if constexpr (TMEM) tmem_free_cta<TCOLS>(tbase, warp);
}


// ================================================================ dual-residue variant (four products, tap kernels)
// The Q residue CTAs of a channel each repeat the whole gather (C3: 28 % of warp time, DRAM 2.2x algorithmic).
// Here one CTA runs TWO column residues l2 = 2u, 2u + 1 from ONE gather: per batch of F2 = 2 pairs it grids once,
// row-transforms every row twice (the four tasks (h, residue) of a row sit in adjacent lanes: both residues load
// the gathered row, __syncwarp, residue 0 stores in place and residue 1 into a second plane set), and runs the
// column pass + products for residue 0 and then residue 1, each with its own accumulators in tensor memory
// (2 x 64 columns per thread).  Per frame and residue the gather work halves; everything else is unchanged:
// 4 column tasks per thread and batch, the same table-read amortisation (2 frames x 2 residues), two CTAs per SM.
constexpr int F2 = 2;  // pairs per batch

template <int NB>
__device__ __forceinline__ void row_task_dual(const float4* __restrict__ src, float4* __restrict__ dst,
                                              const float4* __restrict__ tw, int h, bool valid) {
  C2 z[16];
  transform32<NB>(z, src, 1, tw);
  __syncwarp();  // both residues (and both h) of the row have loaded it: residue 0 may overwrite it
  if (valid) {
#pragma unroll
    for (int k = 0; k < 16; ++k) dst[2 * k + h] = make_float4(z[k].re.x, z[k].re.y, z[k].im.x, z[k].im.y);
  }
}

// one or two products: accumulators (|A_lo|^2, |A_hi|^2) of a thread's 16 pixels in 32 columns of tensor memory
template <int NB>
__device__ __forceinline__ void col_task_tmem2(const float4* __restrict__ col, const float4* __restrict__ tw, uint32_t taddr) {
  C2 z[16];
  uint32_t r[2][16];
  tmem_ld16_issue(taddr, r[0]);  // the first 8 pixels' accumulators travel during the transform
  transform32<NB>(z, col, HS, tw);
#pragma unroll
  for (int c = 0; c < 2; ++c) {
    tmem_wait_ld();
    if (c == 0) tmem_ld16_issue(taddr + 16, r[1]);  // the other 8, during this update
    float a[16];
#pragma unroll
    for (int kk = 0; kk < 8; ++kk) {
      const C2& v = z[8 * c + kk];
      float2 p = make_float2(__uint_as_float(r[c][2 * kk]), __uint_as_float(r[c][2 * kk + 1]));
      p = __ffma2_rn(v.re, v.re, p);
      p = __ffma2_rn(v.im, v.im, p);
      a[2 * kk] = p.x; a[2 * kk + 1] = p.y;
    }
    tmem_st16(taddr + 16 * c, a);
  }
  tmem_wait_st();
}

// partial sums of split units, as epic_fused_fixup, for units of two residues: [cta][slot][residue][4][16][NT]
template <int Q, int NPROD, int NRES>
__global__ void __launch_bounds__(64 * Q) epic_fused_dual_fixup(FusedParams P, int main_grid) {
  // one CTA per (unit, residue): with NRES = 4 a unit is a whole channel and every unit is split between CTAs of the
  // main kernel, so this kernel touches every pixel; (unit, residue) CTAs give it 4x the parallelism of one CTA per
  // unit (measured 0.19 -> see profiles/r02_fused_c2_c3_ncu.md)
  constexpr int NT = 64 * Q, KPT = 16, N = 32 * Q, NACC = NPROD == 4 ? 4 : (NPROD == 2 ? 2 : 1);
  const int unit = blockIdx.x / NRES, res = blockIdx.x - unit * NRES;
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  const long long G = main_grid, first = (long long)unit * P.nb, last = first + P.nb - 1;
  const int b_lo = (int)(((first + 1) * G - 1) / P.total), b_hi = (int)(((last + 1) * G - 1) / P.total);
  if (b_lo == b_hi) return;  // the unit ran in one CTA and was added directly
  const int l1 = (warp & 1) * 16 + (lane >> 1);
  const int rho = (warp >> 1) * 2 + (lane & 1);
  const int c = unit / (Q / NRES), u2 = unit - c * (Q / NRES);
  const size_t plane = (size_t)N * N;
  float* o = P.out + (size_t)c * P.n_planes * plane + (Q * l1 + NRES * u2 + res) + (size_t)rho * N;
  float v[KPT][NACC];
#pragma unroll
  for (int k = 0; k < KPT; ++k)
#pragma unroll
    for (int q = 0; q < NACC; ++q) v[k][q] = 0.0f;
  for (int b = b_lo; b <= b_hi; ++b) {  // in CTA order: the sum does not depend on scheduling
    const int slot = (first <= P.total * b / G) ? 0 : 1;  // does the segment start the CTA's range?
    const float* part = P.partial + ((size_t)((b * 2 + slot) * NRES + res) * NACC * KPT) * NT + tid;
#pragma unroll
    for (int k = 0; k < KPT; ++k)
#pragma unroll
      for (int q = 0; q < NACC; ++q) v[k][q] += __ldcs(part + (size_t)(q * KPT + k) * NT);
  }
#pragma unroll
  for (int k = 0; k < KPT; ++k) add_pixel<NPROD>(o + (size_t)k * 2 * Q * N, plane, v[k]);
}

// NRES residues per CTA: 2, or all 4 (Q = 4, one or two products: 4 x 32 accumulator columns per thread) with one
// pair per batch; the work per batch is the same 4 (pair, residue) column tasks per thread either way.
// PC: every channel has its own cell table (per-channel plans, reading Q15): the thread's cell records are
// reloaded when the work list crosses into the next channel (a separate instantiation, as for the single-residue kernel).
template <int Q, int NPROD, bool DELTA, int NB, bool STG, int NRES, bool PC = false>
__global__ void __launch_bounds__(64 * Q, 2) epic_fused_dual_kernel(FusedParams P) {
  static_assert(!(STG && (DELTA || PC)), "staged tables: tap kernels of one-layout plans only");
  static_assert(NRES == 2 || (NRES == 4 && Q == 4 && NPROD != 4), "four residues: Q = 4, accumulators of 32 columns");
  constexpr int NT = 64 * Q, N = 32 * Q, HQ = Q / NRES, NACC = NPROD == 4 ? 4 : (NPROD == 2 ? 2 : 1);
  constexpr int FB = 4 / NRES;               // pairs per batch
  constexpr int CPT = NPROD == 4 ? 64 : 32;  // accumulator columns per thread and residue
  // Residue r's planes start SET cells after residue r-1's: FB planes plus a skew of 8 / NRES cells.  In the row pass
  // the (h, residue) tasks of a row are adjacent lanes; without the skew the residues' stores of one row fall in the
  // same 16-byte bank groups (216 M of 445 M store wavefronts were conflicts before it)
  constexpr int SET = FB * PLANE + 8 / NRES;
  extern __shared__ __align__(16) unsigned char smem_raw[];
  float4* gA = reinterpret_cast<float4*>(smem_raw);  // [NRES] x [FB][32][HS]: set 0 holds the gridded planes, then residue 0's rows (in place)
  float4* tws = gA + NRES * SET;                     // [2Q][TWV]
  float4* E = tws + 2 * Q * TWV;                     // [FB][A]
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;

  const long long g0 = P.total * (long long)blockIdx.x / gridDim.x;
  const long long g1 = P.total * (long long)(blockIdx.x + 1) / gridDim.x;
  if (g0 >= g1) return;
  constexpr int TCOLS1 = (Q == 4 ? 2 : 1) * CPT, TCOLS = NRES * TCOLS1;  // one block of accumulator columns per residue

  int unit = (int)(g0 / P.nb);  // unit = (channel, group of NRES residues)
  uint2 info[S * S / NT];
#pragma unroll
  for (int j = 0; j < S * S / NT; ++j)
    info[j] = __ldg(P.cell_info + (PC ? (size_t)(unit / HQ) * (S * S) : (size_t)0) + tid + j * NT);
  for (int i = tid; i < NRES * SET; i += NT) gA[i] = make_float4(0.0f, 0.0f, 0.0f, 0.0f);  // rows >= R stay zero
  for (int i = tid; i < 2 * Q * TWV; i += NT) tws[i] = __ldg(P.tw + i);
  float2* tap_s = reinterpret_cast<float2*>(E + FB * P.n_ant);
  uint16_t* ant_s = reinterpret_cast<uint16_t*>(tap_s + P.n_ent);
  if constexpr (STG) {
    for (int i = tid; i < P.n_ent; i += NT) { tap_s[i] = __ldg(P.ent_tap + i); ant_s[i] = __ldg(P.ent_ant + i); }
  }
  __syncthreads();

  const int l1 = (warp & 1) * 16 + (lane >> 1);
  const int rho = (warp >> 1) * 2 + (lane & 1);
  __shared__ uint32_t tmem_slot;
  const uint32_t tbase = tmem_alloc_cta<TCOLS>(&tmem_slot, warp);
  const uint32_t taddr = tbase + (((uint32_t)(warp & 3) * 32u) << 16) + (uint32_t)(warp >> 2) * CPT;
  {
    float zero[16];
#pragma unroll
    for (int i = 0; i < 16; ++i) zero[i] = 0.0f;
#pragma unroll
    for (int res = 0; res < NRES; ++res)
#pragma unroll
      for (int c = 0; c < CPT / 16; ++c) tmem_st16(taddr + res * TCOLS1 + 16 * c, zero);
    tmem_wait_st();
  }

  // S6, as in epic_fused_kernel, for both residues of the unit.  Column layout per thread and residue:
  // four products 4 k + {XX, YY, Re XY, Im XY}; one or two products 2 k + {lo, hi}
  auto flush = [&](int unit, bool complete, int slot) {
    const int c = unit / HQ, u2 = unit - c * HQ;
    const size_t plane = (size_t)N * N;
#pragma unroll 1
    for (int res = 0; res < NRES; ++res) {
      float* o = P.out + (size_t)c * P.n_planes * plane + (Q * l1 + NRES * u2 + res);
      float* part = P.partial + ((size_t)((blockIdx.x * 2 + slot) * NRES + res) * NACC * 16) * NT + tid;
      const uint32_t ta = taddr + res * TCOLS1;
      constexpr int PPC = NPROD == 4 ? 4 : 8;  // pixels per 16-column chunk
#pragma unroll
      for (int c4 = 0; c4 < CPT / 16; ++c4) {
        float a[16], zero[16];
        tmem_ld16(ta + 16 * c4, a);
#pragma unroll
        for (int i = 0; i < 16; ++i) zero[i] = 0.0f;
        tmem_st16(ta + 16 * c4, zero);
#pragma unroll
        for (int kk = 0; kk < PPC; ++kk) {
          const int k = PPC * c4 + kk;
          float v[NACC];
          if constexpr (NPROD == 4) {
            v[0] = a[4 * kk]; v[1] = a[4 * kk + 1]; v[2] = a[4 * kk + 2]; v[3] = a[4 * kk + 3];
          } else if constexpr (NPROD == 2) {
            v[0] = a[2 * kk]; v[1] = a[2 * kk + 1];
          } else {
            v[0] = a[2 * kk] + a[2 * kk + 1];
          }
          if (complete) {
            add_pixel<NPROD>(o + (size_t)(2 * Q * k + rho) * N, plane, v);
          } else {
#pragma unroll
            for (int q = 0; q < NACC; ++q) part[(size_t)(q * 16 + k) * NT] = v[q];
          }
        }
      }
      tmem_wait_st();
    }
  };

  int b = (int)(g0 - (long long)unit * P.nb);
  const int first_unit = unit;
  int seg_begin = b;
  PrefetchSlots ps;
  prefetch_init<NT, FB>(P, tid, ps);
  uint32_t wlo[MAXW], whi[MAXW];
  prefetch_batch<NT, FB>(P, ps, unit / HQ, b, wlo, whi);
  unpack_batch<DELTA>(P, ps, E, wlo, whi, unit / HQ);
  __syncthreads();

  const int ntask = FB * P.R * 2 * NRES;  // (pair, row, h, residue), residue fastest: a row's tasks are adjacent lanes of one warp
  for (long long g = g0; g < g1; ++g) {
    int unit_n = unit, b_n = b + 1;
    if (b_n == P.nb) { b_n = 0; ++unit_n; }
    const bool more = g + 1 < g1;
    if (more) prefetch_batch<NT, FB>(P, ps, unit_n / HQ, b_n, wlo, whi);

    gather_batch<NT, DELTA, STG, DELTA, FB>(P, E, gA, info, ant_s, tap_s);
    __syncthreads();

    const int l2a = NRES * (unit % HQ);
    for (int base = warp * 32; base < ntask; base += NT) {
      const int task = base + lane;
      const bool valid = task < ntask;
      // idle lanes transform the all-zero row 31 of plane 0 (they exist only when R < 32)
      int f = 0, y = S - 1, h = 0, res = 0;
      if (valid) { res = task % NRES; h = (task / NRES) & 1; const int p = task / (2 * NRES); f = p / P.R; y = p - f * P.R; }
      const float4* src = gA + f * PLANE + y * HS;
      row_task_dual<NB>(src, gA + res * SET + f * PLANE + y * HS, tws + (l2a + res + Q * h) * TWV, h, valid);
    }
    __syncthreads();

    if (more) unpack_batch<DELTA>(P, ps, E, wlo, whi, unit_n / HQ);  // E was last read by this batch's gather
#pragma unroll 1
    for (int rf = 0; rf < NRES * FB; ++rf) {
      const int res = rf / FB, f = rf - res * FB;
      int tw_off = rho * TWV;
      asm volatile("" : "+r"(tw_off));
      if constexpr (NPROD == 4) col_task_tmem<NB>(gA + res * SET + f * PLANE + l1, tws + tw_off, taddr + res * TCOLS1);
      else col_task_tmem2<NB>(gA + res * SET + f * PLANE + l1, tws + tw_off, taddr + res * TCOLS1);
    }

    if (unit_n != unit || !more) {
      flush(unit, seg_begin == 0 && b == P.nb - 1, unit == first_unit ? 0 : 1);
      seg_begin = 0;
    }
    if constexpr (PC) {
      if (unit_n / HQ != unit / HQ && more) {  // the next channel's cells (this batch's gather is done with these)
#pragma unroll
        for (int j = 0; j < S * S / NT; ++j)
          info[j] = __ldg(P.cell_info + (size_t)(unit_n / HQ) * (S * S) + tid + j * NT);
      }
    }
    unit = unit_n; b = b_n;
    __syncthreads();  // next batch's E is complete; the planes are free
  }
  tmem_free_cta<TCOLS>(tbase, warp);
}

template <int Q>
size_t fused_dual_smem_bytes(int n_ant, int nres = 2) {
  const int fb = 4 / nres;
  return ((size_t)nres * (fb * PLANE + 8 / nres) + (size_t)2 * Q * TWV + (size_t)fb * n_ant) * sizeof(float4);
}

// ================================================================ tensor-core column pass
// The column transform of a unit is a dense contraction: A[m][(f, pol, l1)] = sum_y F[m][y] H[y][(f, pol, l1)],
// F[m][y] = exp(+2 pi i m y / N) (128 x 32), H = the row-pass output of the batch (32 x 256).  Here it
// runs on the 5th-generation tensor cores (tcgen05.mma, BF16 in, FP32 accumulators in tensor memory)
// instead of the pruned FFT: complex = 4 real products, and to hold the 1e-4 image tolerance every
// operand is split hi + lo in BF16 (16 mantissa bits) with the lo x lo term dropped:
//
//   D_r = Fr Hr - Fi Hi,  D_i = Fi Hr + Fr Hi,  X Y ~ X_hi Y_hi + X_hi Y_lo + X_lo Y_hi
//
// = 24 MMAs of M 128 x N 256 x K 16 per batch (12 per accumulator; the minus sign is the
// instruction's negate-A bit), issued by one thread, asynchronously: they run while the CTA
// gathers and row-transforms the NEXT batch.  gather / rows / unpack are the fused kernel's.
//   convert   row-pass output (fp32, gh) -> four BF16 operands Hr_hi, Hr_lo, Hi_hi, Hi_lo in the
//             K-major core-matrix layout (epic_packed.cuh), 16-byte stores
//   issue     one thread: 24 x tcgen05.mma + tcgen05.commit -> mbarrier
//   epilogue  (one batch later) thread = (image row m = TMEM lane, 16 columns l1): tcgen05.ld of
//             D_r / D_i, S5 products, S6 accumulation in registers
// One CTA per SM (185 KB of shared memory, all 512 TMEM columns).
constexpr int TC_N = 128, TC_NT = 512, TC_NG = F * 2 * S;  // image side, threads, GEMM N = (pair, pol, l1)
constexpr int TC_EPI_NT = 256;                               // threads of the epilogue role (warps 8-15)
constexpr int TC_KPT = TC_N * S / TC_EPI_NT;                 // image pixels per epilogue thread (16 columns l1 of one row m)
constexpr int TC_A_MAT = 4 * TC_N * 8;                       // bf16 elements of one A matrix: [4 K chunks][128 m][8]
constexpr int TC_B_MAT = 4 * TC_NG * 8;                      // of one B matrix: [4 K chunks][256 n][8]

__device__ __forceinline__ void bf16_split2(float a, float b, uint32_t& hi, uint32_t& lo) {
  __nv_bfloat162 h = __floats2bfloat162_rn(a, b);  // .x = a = lower address
  hi = *reinterpret_cast<uint32_t*>(&h);
  __nv_bfloat162 l = __floats2bfloat162_rn(a - __uint_as_float(hi << 16), b - __uint_as_float(hi & 0xFFFF0000u));
  lo = *reinterpret_cast<uint32_t*>(&l);
}

// gh[f][y][l1] = (re_X, re_Y, im_X, im_Y) -> B matrices 0 Hr_hi, 1 Hr_lo, 2 Hi_hi, 3 Hi_lo at
// [K chunk y / 8][n = f * 64 + pol * 32 + l1][y % 8]
__device__ __forceinline__ void tc_convert(const float4* __restrict__ gh, uint16_t* __restrict__ sB, int tid) {
  for (int item = tid; item < F * S * 4; item += TC_NT) {
    const int l1 = item & 31, j = (item >> 5) & 3, f = item >> 7;
    float v[4][8];
#pragma unroll
    for (int i = 0; i < 8; ++i) {
      const float4 c = gh[f * PLANE + (8 * j + i) * HS + l1];
      v[0][i] = c.x; v[1][i] = c.y; v[2][i] = c.z; v[3][i] = c.w;
    }
#pragma unroll
    for (int q = 0; q < 4; ++q) {
      const int pol = q & 1, ri = q >> 1;
      uint32_t hi[4], lo[4];
#pragma unroll
      for (int e = 0; e < 4; ++e) bf16_split2(v[q][2 * e], v[q][2 * e + 1], hi[e], lo[e]);
      const int n = f * 64 + pol * 32 + l1;
      uint16_t* d = sB + (size_t)(2 * ri) * TC_B_MAT + (size_t)(j * TC_NG + n) * 8;
      *reinterpret_cast<uint4*>(d) = make_uint4(hi[0], hi[1], hi[2], hi[3]);
      *reinterpret_cast<uint4*>(d + TC_B_MAT) = make_uint4(lo[0], lo[1], lo[2], lo[3]);
    }
  }
}

// A matrices 0 Fr_hi, 1 Fr_lo, 2 Fi_hi, 3 Fi_lo; D_r at TMEM columns [0, 256), D_i at [256, 512)
__device__ __forceinline__ void tc_issue(uint32_t sA, uint32_t sB, uint32_t tbase, uint64_t* bar) {
  constexpr uint32_t A_LBO = TC_N * 16, B_LBO = TC_NG * 16, SBO = 128;
  constexpr uint32_t A_BYTES = TC_A_MAT * 2, B_BYTES = TC_B_MAT * 2;
  constexpr uint32_t ID = umma_idesc_bf16(128, TC_NG, false), IDN = umma_idesc_bf16(128, TC_NG, true);
  uint32_t acc = 0u;
  auto term = [&](uint32_t d, uint32_t am, uint32_t bm, uint32_t idesc) {
#pragma unroll
    for (uint32_t s = 0; s < 2; ++s) {  // K = 32 = two K = 16 steps
      umma_bf16(d, umma_desc(sA + am * A_BYTES + s * 2 * A_LBO, A_LBO, SBO),
                umma_desc(sB + bm * B_BYTES + s * 2 * B_LBO, B_LBO, SBO), idesc, acc);
      acc = 1u;
    }
  };
  const uint32_t dr = tbase, di = tbase + 256;
  term(dr, 0, 0, ID); term(dr, 0, 1, ID); term(dr, 1, 0, ID);      //  Fr Hr
  term(dr, 2, 2, IDN); term(dr, 2, 3, IDN); term(dr, 3, 2, IDN);   // -Fi Hi
  acc = 0u;
  term(di, 2, 0, ID); term(di, 2, 1, ID); term(di, 3, 0, ID);      //  Fi Hr
  term(di, 0, 2, ID); term(di, 0, 3, ID); term(di, 1, 2, ID);      //  Fr Hi
  umma_commit(bar);
}

template <int NPROD, int K0>
__device__ __forceinline__ void tc_products(const uint32_t (&rx)[8], const uint32_t (&ry)[8], const uint32_t (&ix)[8],
                                            const uint32_t (&iy)[8], float (&acc)[(NPROD == 4 ? 4 : 2) * TC_KPT]) {
#pragma unroll
  for (int k = 0; k < 8; ++k) {
    const float a = __uint_as_float(rx[k]), b = __uint_as_float(ix[k]);
    const float c = __uint_as_float(ry[k]), d = __uint_as_float(iy[k]);
    acc[K0 + k] = fmaf(a, a, fmaf(b, b, acc[K0 + k]));
    acc[TC_KPT + K0 + k] = fmaf(c, c, fmaf(d, d, acc[TC_KPT + K0 + k]));
    if constexpr (NPROD == 4) {  // XY = A_X conj(A_Y) (reading Q11)
      acc[2 * TC_KPT + K0 + k] = fmaf(a, c, fmaf(b, d, acc[2 * TC_KPT + K0 + k]));
      acc[3 * TC_KPT + K0 + k] = fmaf(b, c, fmaf(-a, d, acc[3 * TC_KPT + K0 + k]));
    }
  }
}

// S5 + S6 from the accumulators in tensor memory: acc[q * KPT + k], q = XX, YY, Re XY, Im XY, k = l1 - KPT cg
template <int NPROD>
__device__ __forceinline__ void tc_epilogue(uint32_t tlane, float (&acc)[(NPROD == 4 ? 4 : 2) * TC_KPT]) {
  static_assert(TC_KPT == 16, "two tcgen05.ld .x8 per quantity below");
  // 8 columns at a time: 32 registers of loads in flight beside the (up to 64) accumulators
#pragma unroll 1
  for (int fh = 0; fh < 2 * F; ++fh) {
    const int f = fh >> 1, k0 = (fh & 1) * 8;
    uint32_t rx[8], ry[8], ix[8], iy[8];
    tmem_ld8_issue(tlane + f * 64 + k0, rx);
    tmem_ld8_issue(tlane + f * 64 + 32 + k0, ry);
    tmem_ld8_issue(tlane + 256 + f * 64 + k0, ix);
    tmem_ld8_issue(tlane + 256 + f * 64 + 32 + k0, iy);
    tmem_wait_ld();
    if (fh & 1) {
      tc_products<NPROD, 8>(rx, ry, ix, iy, acc);
    } else {
      tc_products<NPROD, 0>(rx, ry, ix, iy, acc);
    }
  }
}

__device__ __forceinline__ void cta_sync() { asm volatile("bar.sync 0;\n" ::: "memory"); }

// 512 threads in two roles that share gather / unpack / convert and split the middle of a batch:
// warps 0-7 run the row transforms of batch i while warps 8-15 take batch i-1's accumulators out
// of tensor memory (products, sums, flush).  The roles are two instantiations of one loop, so the
// image accumulators are registers of the epilogue warps only.
template <int NPROD, bool DELTA, int NB>
__global__ void __launch_bounds__(TC_NT, 1) epic_tc_kernel(FusedParams P, const uint4* __restrict__ a_tab) {
  constexpr int Q = 4, NT = TC_NT, N = TC_N, NACC = NPROD == 4 ? 4 : 2;
  extern __shared__ __align__(128) unsigned char smem_raw[];
  float4* gh = reinterpret_cast<float4*>(smem_raw);  // [F][32][HS]
  float4* tws = gh + F * PLANE;                      // [2Q][TWV]
  float4* E = tws + 2 * Q * TWV;                     // [F][A]
  uint16_t* sA = reinterpret_cast<uint16_t*>(
      smem_raw + (((size_t)(F * PLANE + 2 * Q * TWV + F * P.n_ant) * sizeof(float4) + 127) & ~(size_t)127));
  uint16_t* sB = sA + 4 * TC_A_MAT;
  __shared__ uint32_t tmem_slot;
  __shared__ __align__(8) uint64_t bar;
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;

  const long long g0 = P.total * (long long)blockIdx.x / gridDim.x;
  const long long g1 = P.total * (long long)(blockIdx.x + 1) / gridDim.x;
  if (g0 >= g1) return;
  for (int i = tid; i < F * PLANE; i += NT) gh[i] = make_float4(0.0f, 0.0f, 0.0f, 0.0f);  // rows >= R stay zero
  for (int i = tid; i < 2 * Q * TWV; i += NT) tws[i] = __ldg(P.tw + i);
  for (int i = tid; i < 4 * TC_A_MAT / 8; i += NT) reinterpret_cast<uint4*>(sA)[i] = __ldg(a_tab + i);
  if (tid == 0) mbar_init(&bar, 1u);
  fence_smem_to_async_proxy();  // the A operand is read by the tensor cores (async proxy)
  const uint32_t tbase = tmem_alloc_cta<512>(&tmem_slot, warp);  // includes the CTA barrier
  const uint32_t sA_u = (uint32_t)__cvta_generic_to_shared(sA), sB_u = (uint32_t)__cvta_generic_to_shared(sB);

  auto run = [&](auto role) {
    constexpr bool EPI = decltype(role)::value;
    // epilogue role: image row m = TMEM lane (a warp reaches the 32 lanes of quadrant warp % 4),
    // columns l1 = KPT cg + k; etid = thread index among the 256 epilogue threads
    const int etid = tid - TC_EPI_NT, m_row = (warp & 3) * 32 + lane, cg = (warp >> 2) & 1;
    const uint32_t tlane = tbase + ((uint32_t)((warp & 3) * 32) << 16) + (uint32_t)(TC_KPT * cg);
    float acc[EPI ? NACC * TC_KPT : 1];
#pragma unroll
    for (int k = 0; k < (EPI ? NACC * TC_KPT : 1); ++k) acc[k] = 0.0f;

    auto flush = [&](int u, bool complete, int slot) {  // as in epic_fused_kernel, other thread <-> pixel mapping
      if constexpr (EPI) {
        const int c = u / Q, l2 = u - c * Q;
        const size_t plane = (size_t)N * N;
        float* o = P.out + (size_t)c * P.n_planes * plane + (size_t)m_row * N + Q * TC_KPT * cg + l2;
        float* part = P.partial + ((size_t)(blockIdx.x * 2 + slot) * NACC * TC_KPT) * TC_EPI_NT + etid;
#pragma unroll
        for (int k = 0; k < TC_KPT; ++k) {
          float v[NACC];
#pragma unroll
          for (int q = 0; q < NACC; ++q) { v[q] = acc[q * TC_KPT + k]; acc[q * TC_KPT + k] = 0.0f; }
          if (complete) {
            add_pixel<NPROD>(o + Q * k, plane, v);
          } else {
#pragma unroll
            for (int q = 0; q < NACC; ++q) part[(size_t)(q * TC_KPT + k) * TC_EPI_NT] = v[q];
          }
        }
      }
    };

    int unit = (int)(g0 / P.nb);
    uint2 info[S * S / NT];
#pragma unroll
    for (int j = 0; j < S * S / NT; ++j) info[j] = __ldg(P.cell_info + tid + j * NT);
    int b = (int)(g0 - (long long)unit * P.nb);
    const int first_unit = unit;
    int seg_begin = b;
    PrefetchSlots ps;
    prefetch_init<NT>(P, tid, ps);
    uint32_t wlo[MAXW], whi[MAXW];
    prefetch_batch<NT>(P, ps, unit / Q, b, wlo, whi);
    unpack_batch<DELTA>(P, ps, E, wlo, whi, unit / Q);
    cta_sync();

    // the batch whose MMAs are in flight: its epilogue (and its unit's flush) happen one iteration later
    bool pend = false, pend_flush = false, pend_complete = false;
    int pend_unit = 0, pend_slot = 0;
    uint32_t phase = 0u;
    auto retire = [&]() {
      if constexpr (EPI) {
        mbar_wait(&bar, phase);
        phase ^= 1u;
        tc_fence_after_sync();
        tc_epilogue<NPROD>(tlane, acc);
        if (pend_flush) flush(pend_unit, pend_complete, pend_slot);
        tc_fence_before_sync();
      }
      pend = false;
    };

    const int ntask = F * P.R * 2;
    for (long long g = g0; g < g1; ++g) {
      int unit_n = unit, b_n = b + 1;
      if (b_n == P.nb) { b_n = 0; ++unit_n; }
      const bool more = g + 1 < g1;
      if (more) prefetch_batch<NT>(P, ps, unit_n / Q, b_n, wlo, whi);

      gather_batch<NT, DELTA, false, DELTA>(P, E, gh, info);
      cta_sync();

      if constexpr (!EPI) {
        const int l2 = unit % Q;
        for (int base = warp * 32; base < ntask; base += TC_NT - TC_EPI_NT) {
          const int task = base + lane;
          const bool valid = task < ntask;
          int f = 0, y = S - 1, h = 0;
          if (valid) { h = task & 1; const int p = task >> 1; f = p / P.R; y = p - f * P.R; }
          row_task<NB>(gh + f * PLANE + y * HS, tws + (l2 + Q * h) * TWV, h, valid);
        }
      } else {
        if (pend) retire();  // the previous batch: D -> products -> registers; frees D for the next MMAs
      }
      pend = false;
      cta_sync();

      if (more) unpack_batch<DELTA>(P, ps, E, wlo, whi, unit_n / Q);  // E was last read by this batch's gather
      tc_convert(gh, sB, tid);                                  // B was last read by the MMAs retired above
      fence_smem_to_async_proxy();
      cta_sync();  // B complete; gh is free for the next gather
      if (tid == 0) {
        tc_fence_after_sync();
        tc_issue(sA_u, sB_u, tbase, &bar);
      }
      pend = true;
      pend_unit = unit;
      pend_flush = unit_n != unit || !more;
      pend_complete = seg_begin == 0 && b == P.nb - 1;
      pend_slot = unit == first_unit ? 0 : 1;
      if (pend_flush) seg_begin = 0;
      unit = unit_n; b = b_n;
    }
    if (pend) retire();
  };
  if (warp < (TC_NT - TC_EPI_NT) / 32) run(std::false_type{});
  else run(std::true_type{});
  tmem_free_cta<512>(tbase, warp);
}

struct FusedTables {
  uint2* cell_info;
  float4* tw;
  uint4* a_tab;  // tensor-core path: the DFT matrix as BF16 hi/lo operands (Q = 4 only), or nullptr
  uint32_t max_cnt;  // most gather entries in one cell
};

template <int Q>
size_t fused_smem_bytes(int n_ant, int ff = F) {
  return ((size_t)ff * PLANE + (size_t)2 * Q * TWV + (size_t)ff * n_ant) * sizeof(float4);
}

inline size_t fused_stage_bytes(int n_ent) { return ((size_t)n_ent * (sizeof(float2) + sizeof(uint16_t)) + 15) & ~(size_t)15; }

template <int Q, int NPROD, bool DELTA, int NB, bool PC, bool STG = false, int FF = F>
int launch_fused(const epic_plan* p, const FusedParams& P, cudaStream_t s) {
  constexpr int NT = 64 * Q;
  const size_t smem = fused_smem_bytes<Q>(P.n_ant, FF) + (STG ? fused_stage_bytes(P.n_ent) : 0);
  auto kern = epic_fused_kernel<Q, NPROD, DELTA, NB, PC, STG, FF>;
  if (smem > 48 * 1024)
    EPIC_CUDA_TRY(cudaFuncSetAttribute((const void*)kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
  int per_sm = 0;
  EPIC_CUDA_TRY(cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, kern, NT, smem));
  if (per_sm < 1) return EPIC_ERR_RANGE;
  // The occupancy query answers 1 for the kernels that allocate tensor memory, although two CTAs
  // (128 of the 512 columns each, 128 registers, 2 x 88 KB) do share an SM: measured 22.1 M frames/s
  // on C3 with 296 CTAs against 18.6 M with 148.  CTAs never wait on one another, so a grid larger
  // than what is resident would only run as two waves.
  if (NPROD == 4 && 2 * (smem + 1024) <= (size_t)227 * 1024) per_sm = std::max(per_sm, 2);
  const long long slots = (long long)per_sm * p->n_sm;
  const int grid = (int)std::min<long long>(P.total, slots);
  constexpr int NACC = NPROD == 4 ? 4 : (NPROD == 2 ? 2 : 1);
  if ((size_t)grid * 2 * NACC * 16 * NT * sizeof(float) > p->scratch_bytes) return EPIC_ERR_RANGE;
  kern<<<grid, NT, smem, s>>>(P);
  epic_fused_fixup<Q, NPROD><<<(unsigned)(P.total / P.nb), NT, 0, s>>>(P, grid);
  EPIC_CUDA_TRY(cudaGetLastError());
  return EPIC_OK;
}

// dual-residue kernel (one layout): sized for two CTAs per SM
template <int Q, int NPROD, bool DELTA, int NB, bool STG, int NRES = 2, bool PC = false>
int launch_fused_dual(const epic_plan* p, FusedParams P, cudaStream_t s) {
  constexpr int NT = 64 * Q, NACC = NPROD == 4 ? 4 : (NPROD == 2 ? 2 : 1), FB = 4 / NRES;
  P.pairs_per_batch = FB;
  const int per_batch = P.n_pol == 2 ? FB : 2 * FB;  // time samples per batch
  P.nb = (P.n_t + per_batch - 1) / per_batch;
  P.total = (long long)P.n_chan * (Q / NRES) * P.nb;
  const size_t smem = fused_dual_smem_bytes<Q>(P.n_ant, NRES) + (STG ? fused_stage_bytes(P.n_ent) : 0);
  auto kern = epic_fused_dual_kernel<Q, NPROD, DELTA, NB, STG, NRES, PC>;
  if (smem > 48 * 1024)
    EPIC_CUDA_TRY(cudaFuncSetAttribute((const void*)kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
  // tensor-memory kernels: the occupancy query answers 1; two CTAs (at most 2 x 256 of the 512 columns) share an SM
  const int per_sm = 2 * (smem + 1024) <= (size_t)227 * 1024 ? 2 : 1;
  const int grid = (int)std::min<long long>(P.total, (long long)per_sm * p->n_sm);
  if ((size_t)grid * 2 * NRES * NACC * 16 * NT * sizeof(float) > p->scratch_bytes) return EPIC_ERR_RANGE;
  kern<<<grid, NT, smem, s>>>(P);
  epic_fused_dual_fixup<Q, NPROD, NRES><<<(unsigned)(P.total / P.nb) * NRES, NT, 0, s>>>(P, grid);
  EPIC_CUDA_TRY(cudaGetLastError());
  return EPIC_OK;
}

template <int Q, int NPROD, bool DELTA>
int launch_fused_nb(const epic_plan* p, const FusedParams& P, cudaStream_t s) {
  // elements y + 16 of a row/column are read only while y < NB (the rest of the block is empty)
  const bool pc = P.cell_stride != 0, nb12 = std::max(p->R, p->Cc) <= 16 + 12;
  if constexpr (Q == 1) {  // N = 32: a single residue per axis, so no residue groups; one instantiation per layout kind
    // two pairs per batch: the 64 threads' prefetch slots then hold up to 256 antennas
    return pc ? launch_fused<1, NPROD, DELTA, 16, true, false, F2>(p, P, s) : launch_fused<1, NPROD, DELTA, 16, false, false, F2>(p, P, s);
  } else {
    // NR residues per CTA from one gather (epic_fused_dual_kernel): all four of a channel when the
    // accumulators are 32 columns per residue (Q = 4, one or two products; C2 32.3 -> 33.5 M frames/s over two), else
    // two.  Its shared memory is never more than the single-residue kernel's (same planes, fewer voltages), so it fits
    // whenever fused_supported said yes.
    constexpr int NR = (Q == 4 && NPROD != 4) ? 4 : 2;
    if (pc)  // one layout per channel: the instantiation that reloads its cell records when the channel changes
      return nb12 ? launch_fused_dual<Q, NPROD, DELTA, 12, false, NR, true>(p, P, s)
                  : launch_fused_dual<Q, NPROD, DELTA, 16, false, NR, true>(p, P, s);
    if constexpr (!DELTA) {  // staged gather tables, if two CTAs still fit an SM with them
      if (2 * (fused_dual_smem_bytes<Q>(P.n_ant, NR) + fused_stage_bytes(P.n_ent) + 1024 + 128) <= (size_t)227 * 1024)
        return nb12 ? launch_fused_dual<Q, NPROD, false, 12, true, NR>(p, P, s) : launch_fused_dual<Q, NPROD, false, 16, true, NR>(p, P, s);
    }
    return nb12 ? launch_fused_dual<Q, NPROD, DELTA, 12, false, NR>(p, P, s) : launch_fused_dual<Q, NPROD, DELTA, 16, false, NR>(p, P, s);
  }
}

template <int Q>
int launch_fused_q(const epic_plan* p, const FusedParams& P, int n_products, cudaStream_t s) {
  // The delta instantiations gather in integers (gather_batch EB): no delay phasors, at most 16 antennas
  // in a cell.  Other delta plans run the tap kernels with their unit taps (1 + 0i), which is exact too.
  const FusedTables* ft = static_cast<const FusedTables*>(p->d_fused);
  const bool delta = p->t.is_delta != 0 && P.phasor == nullptr && ft->max_cnt <= 16u;
#ifdef EPIC_FUSED_DEV_ONE  // development builds: compile a single instantiation
  if (Q == 4 && n_products == 2 && delta) return launch_fused_dual<4, 2, true, 12, false, 4>(p, P, s);
  return EPIC_ERR_RANGE;
#else
  switch (n_products) {
    case 1: return delta ? launch_fused_nb<Q, 1, true>(p, P, s) : launch_fused_nb<Q, 1, false>(p, P, s);
    case 2: return delta ? launch_fused_nb<Q, 2, true>(p, P, s) : launch_fused_nb<Q, 2, false>(p, P, s);
    default: return delta ? launch_fused_nb<Q, 4, true>(p, P, s) : launch_fused_nb<Q, 4, false>(p, P, s);
  }
#endif
}

}  // namespace

// ---------------------------------------------------------------- host side
int fused_plan_init(epic_plan* p) {
  p->fused_ok = 0;
  p->d_fused = nullptr;
  const int Q = p->N / S;
  if (p->N % S != 0 || (Q != 1 && Q != 2 && Q != 4)) return EPIC_OK;  // N = 32 (no padding beyond the block), 64, 128
  if (p->R > S || p->Cc > S) return EPIC_OK;
  if (p->h_ent_ant.size() >= ((size_t)1 << 24)) return EPIC_OK;
  // one table of S x S cell records per layout (channel c of a per-channel plan reads table c)
  std::vector<uint2> info;
  for (int l = 0; l < p->n_layout; ++l) {
    std::vector<uint32_t> dense((size_t)S * S, 0u);
    for (uint32_t i = p->h_cell_off[l]; i < p->h_cell_off[l + 1]; ++i) {
      const CellRec& c = p->h_cells[i];
      if (c.ent_count > 255u) return EPIC_OK;  // falls back to the two-pass path
      dense[(size_t)c.y * S + c.x] = (c.ent_begin << 8) | c.ent_count;
    }
    // every cell of the R x 32 block (columns >= Cc are re-zeroed each batch: the row pass writes
    // its output in place), sorted by entry count so that warps see uniform trip counts
    // (tap plans: the plan builder has already chosen the order, bank-aware within equal counts)
    std::vector<uint2> li;
    const size_t n_slots = (size_t)p->R * S;
    if (p->h_slot_order.size() == (size_t)p->n_layout * n_slots) {
      for (size_t i = 0; i < n_slots; ++i) {
        const uint32_t s = p->h_slot_order[(size_t)l * n_slots + i], y = s / S, x = s % S;
        li.push_back(make_uint2(dense[s], (uint32_t)(y * HS + x)));
      }
    } else {
      for (int y = 0; y < p->R; ++y)
        for (int x = 0; x < S; ++x) li.push_back(make_uint2(dense[(size_t)y * S + x], (uint32_t)(y * HS + x)));
      std::stable_sort(li.begin(), li.end(),
                       [](const uint2& a, const uint2& b) { return (a.x & 0xFFu) > (b.x & 0xFFu); });
    }
    li.resize((size_t)S * S, make_uint2(0u, 0xFFFFFFFFu));
    info.insert(info.end(), li.begin(), li.end());
  }
  // TwSet of every residue rho = 0..2Q-1, from double (reading Q8: + sign): r = exp(2 pi i rho / N)
  std::vector<float4> tw((size_t)2 * Q * TWV);
  for (int rho = 0; rho < 2 * Q; ++rho) {
    auto cis = [&](double r_pow, int k, int n, float* re, float* im) {  // r^r_pow W_n^k
      const double ang = 2.0 * M_PI * ((double)rho * r_pow / (double)p->N + (double)k / (double)n);
      *re = (float)std::cos(ang);
      *im = (float)std::sin(ang);
    };
    float v[20] = {0};
    cis(16.0, 0, 1, &v[0], &v[1]);                                       // fold: r^16
    cis(8.0, 0, 2, &v[2], &v[3]);                                        // level 2
    cis(4.0, 0, 4, &v[4], &v[5]);                                        // level 4
    for (int k = 0; k < 2; ++k) cis(2.0, k, 8, &v[6 + 2 * k], &v[7 + 2 * k]);    // level 8
    for (int k = 0; k < 4; ++k) cis(1.0, k, 16, &v[10 + 2 * k], &v[11 + 2 * k]);  // level 16
    for (int j = 0; j < TWV; ++j)
      tw[(size_t)rho * TWV + j] = make_float4(v[4 * j], v[4 * j + 1], v[4 * j + 2], v[4 * j + 3]);
  }
  // tensor-core path (Q = 4): F[m][y] = exp(+2 pi i m y / N), m < 128, y < 32, from double, split
  // hi + lo in BF16; matrices Fr_hi, Fr_lo, Fi_hi, Fi_lo, each [K chunk y / 8][m][y % 8]
  std::vector<uint16_t> a_tab;
  if (Q == 4) {
    auto bf16_rn = [](float v) {
      uint32_t u;
      std::memcpy(&u, &v, 4);
      return (uint16_t)((u + 0x7FFFu + ((u >> 16) & 1u)) >> 16);
    };
    auto bf16_f = [](uint16_t h) {
      const uint32_t u = (uint32_t)h << 16;
      float f;
      std::memcpy(&f, &u, 4);
      return f;
    };
    a_tab.assign((size_t)4 * TC_A_MAT, 0);
    for (int m = 0; m < TC_N; ++m)
      for (int y = 0; y < S; ++y) {
        const double ang = 2.0 * M_PI * (double)((m * y) % p->N) / (double)p->N;
        const double v[2] = {std::cos(ang), std::sin(ang)};
        for (int ri = 0; ri < 2; ++ri) {
          const uint16_t hi = bf16_rn((float)v[ri]);
          const uint16_t lo = bf16_rn((float)(v[ri] - (double)bf16_f(hi)));
          const size_t at = ((size_t)(y >> 3) * TC_N + m) * 8 + (y & 7);
          a_tab[(size_t)(2 * ri) * TC_A_MAT + at] = hi;
          a_tab[(size_t)(2 * ri + 1) * TC_A_MAT + at] = lo;
        }
      }
  }
  FusedTables* ft = new (std::nothrow) FusedTables();
  if (!ft) return EPIC_ERR_NOMEM;
  ft->cell_info = nullptr;
  ft->tw = nullptr;
  ft->a_tab = nullptr;
  ft->max_cnt = 0;
  for (const CellRec& c : p->h_cells) ft->max_cnt = std::max(ft->max_cnt, c.ent_count);
  cudaError_t ce = cudaMalloc(&ft->cell_info, info.size() * sizeof(uint2));
  if (ce == cudaSuccess) ce = cudaMalloc(&ft->tw, tw.size() * sizeof(float4));
  if (ce == cudaSuccess && !a_tab.empty()) {
    ce = cudaMalloc(&ft->a_tab, a_tab.size() * sizeof(uint16_t));
    if (ce == cudaSuccess) ce = cudaMemcpy(ft->a_tab, a_tab.data(), a_tab.size() * sizeof(uint16_t), cudaMemcpyHostToDevice);
  }
  if (ce == cudaSuccess)
    ce = cudaMemcpy(ft->cell_info, info.data(), info.size() * sizeof(uint2), cudaMemcpyHostToDevice);
  if (ce == cudaSuccess) ce = cudaMemcpy(ft->tw, tw.data(), tw.size() * sizeof(float4), cudaMemcpyHostToDevice);
  if (ce != cudaSuccess) {
    set_cuda_error(ce);
    if (ft->cell_info) cudaFree(ft->cell_info);
    if (ft->tw) cudaFree(ft->tw);
    if (ft->a_tab) cudaFree(ft->a_tab);
    delete ft;
    return ce == cudaErrorMemoryAllocation ? EPIC_ERR_NOMEM : EPIC_ERR_CUDA;
  }
  p->d_fused = ft;
  p->fused_ok = 1;
  return EPIC_OK;
}

void fused_plan_free(epic_plan* p) {
  FusedTables* ft = static_cast<FusedTables*>(p->d_fused);
  if (ft) {
    if (ft->cell_info) cudaFree(ft->cell_info);
    if (ft->tw) cudaFree(ft->tw);
    if (ft->a_tab) cudaFree(ft->a_tab);
    delete ft;
  }
  p->d_fused = nullptr;
  p->fused_ok = 0;
}

int fused_supported(const epic_plan* p, int is_cf32, int n_pol, int n_products) {
  if (!p->fused_ok && p->wide_ok) return wide_supported(p, is_cf32, n_pol, n_products);  // support beyond 32 x 32
  if (!p->fused_ok || is_cf32) return 0;
  if (!((n_pol == 1 && n_products == 1) || (n_pol == 2 && (n_products == 2 || n_products == 4)))) return 0;
  const int Q = p->N / S;
  const int nt = 64 * Q;
  const int a_pad = (p->n_ant + 3) & ~3;  // a short tail group is fetched as bytes (prefetch_batch)
  if (Q == 1) {  // N = 32: one residue per axis, the single-residue kernel with 64 threads
    if ((long long)F2 * (a_pad / 4) > (long long)MAXW * nt) return 0;
    return fused_smem_bytes<1>(a_pad, F2) <= (size_t)200 * 1024 ? 1 : 0;
  }
  if ((long long)F2 * (a_pad / 4) > (long long)MAXW * nt) return 0;  // prefetch registers (at most F2 pairs per batch)
  const size_t smem = Q == 2 ? fused_dual_smem_bytes<2>(a_pad) : fused_dual_smem_bytes<4>(a_pad);
  return smem <= (size_t)200 * 1024 ? 1 : 0;
}

static size_t tc_smem_bytes(int n_ant) {
  const size_t head = ((size_t)F * PLANE + (size_t)2 * 4 * TWV + (size_t)F * n_ant) * sizeof(float4);
  return ((head + 127) & ~(size_t)127) + (size_t)4 * (TC_A_MAT + TC_B_MAT) * sizeof(uint16_t);
}

int tensor_supported(const epic_plan* p, int is_cf32, int n_pol, int n_products) {
  if (!p->fused_ok || !fused_supported(p, is_cf32, n_pol, n_products)) return 0;
  const FusedTables* ft = static_cast<const FusedTables*>(p->d_fused);
  if (p->N != TC_N || !ft->a_tab || n_pol != 2 || p->n_layout != 1) return 0;
  if ((long long)F * (((p->n_ant + 3) & ~3) / 4) > (long long)MAXW * TC_NT) return 0;  // prefetch registers
  return tc_smem_bytes((p->n_ant + 3) & ~3) <= (size_t)226 * 1024 ? 1 : 0;
}

template <int NPROD, bool DELTA, int NB>
static int launch_tc(const epic_plan* p, const FusedParams& P, const uint4* a_tab, cudaStream_t s) {
  const size_t smem = tc_smem_bytes(P.n_ant);
  auto kern = epic_tc_kernel<NPROD, DELTA, NB>;
  EPIC_CUDA_TRY(cudaFuncSetAttribute((const void*)kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
  const int grid = (int)std::min<long long>(P.total, p->n_sm);  // one CTA per SM (shared memory, all of TMEM)
  constexpr int NACC = NPROD == 4 ? 4 : 2;
  if ((size_t)grid * 2 * NACC * TC_KPT * TC_EPI_NT * sizeof(float) > p->scratch_bytes) return EPIC_ERR_RANGE;
  kern<<<grid, TC_NT, smem, s>>>(P, a_tab);
  epic_fused_fixup<4, NPROD, true><<<(unsigned)(P.total / P.nb), TC_EPI_NT, 0, s>>>(P, grid);
  EPIC_CUDA_TRY(cudaGetLastError());
  return EPIC_OK;
}

static void fill_params(const epic_plan* p, const ImageArgs& a, FusedParams& P) {
  const FusedTables* ft = static_cast<const FusedTables*>(p->d_fused);
  const int Q = p->N / S;
  P.volt = static_cast<const uint8_t*>(a.volt);
  P.out = a.out;
  P.cell_info = ft->cell_info;
  P.cell_stride = p->n_layout > 1 ? S * S : 0;
  P.ent_ant = p->t.ent_ant;
  P.ent_tap = p->t.ent_tap;
  P.tw = ft->tw;
  P.partial = static_cast<float*>(p->d_scratch);
  P.native = a.native;
  P.phasor = a.phasor_pair;
  P.n_t = a.n_t;
  P.n_chan = a.n_chan;
  P.n_ant = (p->n_ant + 3) & ~3;
  P.n_ant_true = p->n_ant;
  // rows that are not word-aligned (antenna count no multiple of 4, or a voltage pointer that is not): bytes
  P.unaligned = (p->n_ant & 3) != 0 || (reinterpret_cast<uintptr_t>(a.volt) & 3u) != 0;
  P.n_ent = p->t.n_ent;
  P.n_pol = a.n_pol;
  P.n_planes = a.n_planes;
  P.R = p->R;
  P.Cc = p->Cc;
  // measured on C2 (R = 25): 5 pairs per batch fill the row pass's 256 lanes (250 instead of 200 tasks) but change
  // nothing (31.3 M against 31.5 M frames/s) -- the SM's other CTA already covers the idle warp; 4 stays
  P.pairs_per_batch = p->N == S ? F2 : F;  // N = 32 runs two pairs per batch (launch_fused_nb)
  const int per_batch = a.n_pol == 2 ? P.pairs_per_batch : 2 * P.pairs_per_batch;  // time samples per batch
  P.nb = (a.n_t + per_batch - 1) / per_batch;
  P.total = (long long)a.n_chan * Q * P.nb;
}

int tensor_image(epic_plan* p, const ImageArgs& a) {
  const FusedTables* ft = static_cast<const FusedTables*>(p->d_fused);
  FusedParams P;
  fill_params(p, a, P);
  // delta instantiations: integer gather, under the conditions of launch_fused_q
  const bool delta = p->t.is_delta != 0 && P.phasor == nullptr && ft->max_cnt <= 16u;
  const bool nb12 = std::max(p->R, p->Cc) <= 16 + 12;
  int st;
#define EPIC_TC_CASE(NPROD, DELTA, NB) st = launch_tc<NPROD, DELTA, NB>(p, P, ft->a_tab, a.stream)
  if (a.n_products == 2) {
    if (delta) { if (nb12) EPIC_TC_CASE(2, true, 12); else EPIC_TC_CASE(2, true, 16); }
    else { if (nb12) EPIC_TC_CASE(2, false, 12); else EPIC_TC_CASE(2, false, 16); }
  } else {
    if (delta) { if (nb12) EPIC_TC_CASE(4, true, 12); else EPIC_TC_CASE(4, true, 16); }
    else { if (nb12) EPIC_TC_CASE(4, false, 12); else EPIC_TC_CASE(4, false, 16); }
  }
#undef EPIC_TC_CASE
  if (st != EPIC_OK) return st;
  p->last_launches = 2;
  return EPIC_OK;
}

int fused_image(epic_plan* p, const ImageArgs& a) {
  if (!p->fused_ok && p->wide_ok) return wide_image(p, a);
  const int Q = p->N / S;
  FusedParams P;
  fill_params(p, a, P);
  int st;
  if (Q == 1) st = launch_fused_q<1>(p, P, a.n_products, a.stream);
  else if (Q == 2) st = launch_fused_q<2>(p, P, a.n_products, a.stream);
  else st = launch_fused_q<4>(p, P, a.n_products, a.stream);
  if (st != EPIC_OK) return st;
  p->last_launches = 2;  // the fused kernel and the (tiny) fix-up of split units
  return EPIC_OK;
}

// ---------------------------------------------------------------- epic_image_noalloc (include/epic.h)
namespace {

// Device address of epic_noalloc_scratch on the CURRENT device, looked up once per device (set-up; no allocation).
constexpr int NOALLOC_MAX_DEVICES = 64;
void* g_noalloc_ptr[NOALLOC_MAX_DEVICES] = {nullptr};
std::mutex g_noalloc_mutex;

int noalloc_scratch_ptr(float** out) {
  int dev = -1;
  EPIC_CUDA_TRY(cudaGetDevice(&dev));
  if (dev < 0 || dev >= NOALLOC_MAX_DEVICES) return EPIC_ERR_RANGE;
  std::lock_guard<std::mutex> lock(g_noalloc_mutex);
  if (!g_noalloc_ptr[dev]) {
    void* q = nullptr;
    EPIC_CUDA_TRY(cudaGetSymbolAddress(&q, epic_noalloc_scratch));  // this device's copy of the array
    if (!q) return EPIC_ERR_CUDA;
    g_noalloc_ptr[dev] = q;
  }
  *out = static_cast<float*>(g_noalloc_ptr[dev]);
  return EPIC_OK;
}

// launch_fused_dual with the static array as the partial-sum scratch: same kernels, same launch configuration, so the
// images are bit-identical to epic_image's.  Nothing in the scratch has to start at zero: the fix-up kernel reads
// exactly the slots the main kernel of the same call wrote (the segments of the units that were split).
template <int Q, int NPROD, bool DELTA, int NB, bool STG, int NRES>
int launch_dual_static(const epic_plan* p, FusedParams P, float* scratch, cudaStream_t s) {
  constexpr int NT = 64 * Q, NACC = NPROD == 4 ? 4 : (NPROD == 2 ? 2 : 1), FB = 4 / NRES;
  P.partial = scratch;
  P.pairs_per_batch = FB;
  const int per_batch = P.n_pol == 2 ? FB : 2 * FB;  // time samples per batch
  P.nb = (P.n_t + per_batch - 1) / per_batch;
  P.total = (long long)P.n_chan * (Q / NRES) * P.nb;
  const size_t smem = fused_dual_smem_bytes<Q>(P.n_ant, NRES) + (STG ? fused_stage_bytes(P.n_ent) : 0);
  auto kern = epic_fused_dual_kernel<Q, NPROD, DELTA, NB, STG, NRES>;
  if (smem > 48 * 1024)
    EPIC_CUDA_TRY(cudaFuncSetAttribute((const void*)kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
  const int per_sm = 2 * (smem + 1024) <= (size_t)227 * 1024 ? 2 : 1;
  const int grid = (int)std::min<long long>(P.total, (long long)per_sm * p->n_sm);
  if ((size_t)grid * 2 * NRES * NACC * 16 * NT * sizeof(float) > EPIC_NOALLOC_SCRATCH_BYTES) return EPIC_ERR_SCRATCH;
  kern<<<grid, NT, smem, s>>>(P);
  epic_fused_dual_fixup<Q, NPROD, NRES><<<(unsigned)(P.total / P.nb) * NRES, NT, 0, s>>>(P, grid);
  EPIC_CUDA_TRY(cudaGetLastError());
  return EPIC_OK;
}

// the choices of launch_fused_nb for one-layout plans
template <int Q, int NPROD, bool DELTA>
int launch_static_nb(const epic_plan* p, const FusedParams& P, float* scratch, cudaStream_t s) {
  const bool nb12 = std::max(p->R, p->Cc) <= 16 + 12;
  constexpr int NR = (Q == 4 && NPROD != 4) ? 4 : 2;
  if constexpr (!DELTA) {
    if (2 * (fused_dual_smem_bytes<Q>(P.n_ant, NR) + fused_stage_bytes(P.n_ent) + 1024 + 128) <= (size_t)227 * 1024)
      return nb12 ? launch_dual_static<Q, NPROD, false, 12, true, NR>(p, P, scratch, s)
                  : launch_dual_static<Q, NPROD, false, 16, true, NR>(p, P, scratch, s);
  }
  return nb12 ? launch_dual_static<Q, NPROD, DELTA, 12, false, NR>(p, P, scratch, s)
              : launch_dual_static<Q, NPROD, DELTA, 16, false, NR>(p, P, scratch, s);
}

// the choices of launch_fused_q
template <int Q>
int launch_static_q(const epic_plan* p, const FusedParams& P, int n_products, float* scratch, cudaStream_t s) {
  const FusedTables* ft = static_cast<const FusedTables*>(p->d_fused);
  const bool delta = p->t.is_delta != 0 && P.phasor == nullptr && ft->max_cnt <= 16u;
#ifdef EPIC_FUSED_DEV_ONE  // development builds: compile a single instantiation
  if (Q == 4 && n_products == 2 && delta) return launch_dual_static<4, 2, true, 12, false, 4>(p, P, scratch, s);
  return EPIC_ERR_RANGE;
#else
  switch (n_products) {
    case 1: return delta ? launch_static_nb<Q, 1, true>(p, P, scratch, s) : launch_static_nb<Q, 1, false>(p, P, scratch, s);
    case 2: return delta ? launch_static_nb<Q, 2, true>(p, P, scratch, s) : launch_static_nb<Q, 2, false>(p, P, scratch, s);
    default: return delta ? launch_static_nb<Q, 4, true>(p, P, scratch, s) : launch_static_nb<Q, 4, false>(p, P, scratch, s);
  }
#endif
}

}  // namespace

long long noalloc_scratch_bytes() { return (long long)EPIC_NOALLOC_SCRATCH_BYTES; }

// The caller (epic_image_noalloc in epic_plan.cu) has checked: fused_ok, one layout, fused_supported.
int fused_image_noalloc(epic_plan* p, const ImageArgs& a) {
  float* scratch = nullptr;
  const int sp = noalloc_scratch_ptr(&scratch);  // set-up: once per device, also on an empty call
  if (sp != EPIC_OK) return sp;
  if (a.n_t == 0 || a.n_chan == 0) return EPIC_OK;
  const int Q = p->N / S;
  FusedParams P;
  fill_params(p, a, P);
  const int st = Q == 2 ? launch_static_q<2>(p, P, a.n_products, scratch, a.stream)
                        : launch_static_q<4>(p, P, a.n_products, scratch, a.stream);
  if (st != EPIC_OK) return st;
  p->last_launches = 2;
  return EPIC_OK;
}

}  // namespace epic
