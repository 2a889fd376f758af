// Wide fused EPIC path: the one-kernel design of epic_fused.cu for apertures whose occupied cells need
// up to 64 x 64 cells (N = 64, 128) -- e.g. the paper's own operating point, 256 antennas in a
// 110 m x 100 m aperture on lambda/2 cells at 55.25 MHz with the 3 m top-hat (PAPER.md:148, 166-168:
// about 43 x 39 cells), which the 32 x 32 kernel cannot hold.  PAPER.md:122-126 steps S1..S6.
//
// Same decomposition: unit = (channel c, column residue l2), image columns l = Q l1 + l2, and for a
// residue rho' the outputs 2 Q k + rho' of a line come from a fold and one 16-point ramped transform.
// With up to 64 cells per line the fold has up to four terms (r = W_N^{rho'}, cells beyond the box are
// structurally zero and never read):
//
//   X[2 Q k + rho'] = sum_{y<16} ( in[y] + r^32 in[y+32] + r^16 (in[y+16] + r^32 in[y+48]) ) r^y W_16^{y k}
//
// Along x the r^32 term is a constant of the unit, r^32 = W_N^{32 l2} = W_Q^{l2} in {1, i, -1, -i}, so
// it is applied in the GATHER: a cell (y, x >= 32) is summed into the folded cell (y, x - 32) times
// W_Q^{l2}.  The shared plane stays 32 cells wide ([rows][34] float4) and the row pass is the
// 32 x 32 kernel's, unchanged.  Along y the column pass folds the up-to-four row blocks while loading.
// Two to four pairs per batch, by plane height (a plane is up to 64 x 34 x 16 B = 34.8 KB), keep two CTAs on an SM.
#include <algorithm>
#include <cmath>
#include <cstring>
#include <new>
#include <vector>

#include "epic_internal.h"
#include "epic_packed.cuh"
#include "epic_fused_core.cuh"

namespace epic {
namespace {


// column fold: z[bitrev(y)] = in[y] + c32 in[y+32] + c16 (in[y+16] + c32 in[y+48]); rows y+32 exist while
// y < NB2, rows y+48 while y < NB3 (RA = 32: neither, 40: NB2 = 8, 48: NB2 = 16, 64: both)
__device__ __forceinline__ void cmac(float2& sr, float2& si, float2 br, float2 bi, float cr, float ci) {
  sr = __ffma2_rn(br, f2(cr), sr); sr = __ffma2_rn(neg2(bi), f2(ci), sr);
  si = __ffma2_rn(bi, f2(cr), si); si = __ffma2_rn(br, f2(ci), si);
}
template <int NB2, int NB3, int Y>
__device__ __forceinline__ void fold_wide(C2 (&z)[16], const float4* __restrict__ in, float c16r, float c16i,
                                          float c32r, float c32i) {
  if constexpr (Y < 16) {
    const float4 a = in[Y * HS];
    float2 sr = make_float2(a.x, a.y), si = make_float2(a.z, a.w);
    if constexpr (Y < NB2) {
      const float4 b = in[(Y + 32) * HS];
      cmac(sr, si, make_float2(b.x, b.y), make_float2(b.z, b.w), c32r, c32i);
    }
    const float4 c = in[(Y + 16) * HS];
    float2 tr = make_float2(c.x, c.y), ti = make_float2(c.z, c.w);
    if constexpr (Y < NB3) {
      const float4 d = in[(Y + 48) * HS];
      cmac(tr, ti, make_float2(d.x, d.y), make_float2(d.z, d.w), c32r, c32i);
    }
    cmac(sr, si, tr, ti, c16r, c16i);
    z[bitrev4(Y)].re = sr; z[bitrev4(Y)].im = si;
    if constexpr ((Y & 1) == 1 && Y < 15) __syncwarp();  // bounds the loads in flight (see fold<> in epic_fused_core.cuh)
    fold_wide<NB2, NB3, Y + 1>(z, in, c16r, c16i, c32r, c32i);
  }
}

// tw[4] = (w16r3, w16i3, r^32.re, r^32.im): the wide kernel's TwSet carries the second fold constant
template <int NB2, int NB3>
__device__ __forceinline__ void transform_wide(C2 (&z)[16], const float4* __restrict__ col, const float4* __restrict__ tw) {
  const float4 t0 = tw[0], t4 = tw[4];
  fold_wide<NB2, NB3, 0>(z, col, t0.x, t0.y, t4.z, t4.w);
  fft16_ramped(z, tw, t0.z, t0.w);
}

template <int NB2, int NB3>
__device__ __forceinline__ void col_task_wide(const float4* __restrict__ col, const float4* __restrict__ tw, float2 (&acc)[16]) {
  C2 z[16];
  transform_wide<NB2, NB3>(z, col, tw);
#pragma unroll
  for (int k = 0; k < 16; ++k) {
    acc[k] = __ffma2_rn(z[k].re, z[k].re, acc[k]);
    acc[k] = __ffma2_rn(z[k].im, z[k].im, acc[k]);
  }
}

// four products: accumulators in tensor memory, as col_task_tmem of the 32 x 32 kernel
template <int NB2, int NB3>
__device__ __forceinline__ void col_task_wide_tmem(const float4* __restrict__ col, const float4* __restrict__ tw, uint32_t taddr) {
  C2 z[16];
  uint32_t r[2][16];
  tmem_ld16_issue(taddr, r[0]);
  transform_wide<NB2, NB3>(z, col, tw);
#pragma unroll
  for (int c = 0; c < 4; ++c) {
    tmem_wait_ld();
    if (c < 3) tmem_ld16_issue(taddr + 16 * (c + 1), r[(c + 1) & 1]);
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

// S3 with the x-fold: every thread owns cell slots tid + j NT of the R x 32 folded block (sorted by entry
// count); a slot's list holds first the entries of cell (y, x), then those of cell (y, x + 32), whose sum
// enters times fx = W_Q^{l2}.  Sums in table order, no atomics.
template <int NT, int PLW, int FW>
__device__ __forceinline__ void gather_wide(const FusedParams& P, const float4* __restrict__ E, float4* __restrict__ gh,
                                            const uint2* __restrict__ info, int n_slot, float fxr, float fxi) {
  for (int s = threadIdx.x; s < n_slot; s += NT) {
    const uint2 ci = info[s];
    const uint32_t beg = ci.x >> 8, n_lo = ci.x & 0xFFu, n_hi = ci.y >> 16;
    float2 sr[FW], si[FW], hr[FW], hi[FW];
#pragma unroll
    for (int f = 0; f < FW; ++f) {
      sr[f] = make_float2(0.0f, 0.0f); si[f] = make_float2(0.0f, 0.0f);
      hr[f] = make_float2(0.0f, 0.0f); hi[f] = make_float2(0.0f, 0.0f);
    }
    for (uint32_t e = beg; e < beg + n_lo; ++e) {
      const float4* ea = E + __ldg(P.ent_ant + e);
      const float2 w = __ldg(P.ent_tap + e);
#pragma unroll
      for (int f = 0; f < FW; ++f) {
        const float4 v = ea[f * P.n_ant];
        cmac(sr[f], si[f], make_float2(v.x, v.y), make_float2(v.z, v.w), w.x, w.y);
      }
    }
    for (uint32_t e = beg + n_lo; e < beg + n_lo + n_hi; ++e) {
      const float4* ea = E + __ldg(P.ent_ant + e);
      const float2 w = __ldg(P.ent_tap + e);
#pragma unroll
      for (int f = 0; f < FW; ++f) {
        const float4 v = ea[f * P.n_ant];
        cmac(hr[f], hi[f], make_float2(v.x, v.y), make_float2(v.z, v.w), w.x, w.y);
      }
    }
    float4* dst = gh + (ci.y & 0xFFFFu);
#pragma unroll
    for (int f = 0; f < FW; ++f) {
      if (n_hi) cmac(sr[f], si[f], hr[f], hi[f], fxr, fxi);
      dst[f * PLW] = make_float4(sr[f].x, sr[f].y, si[f].x, si[f].y);
    }
  }
}

// RA: rows allocated per plane (32, 40, 48 or 64 >= R; rows R .. RA-1 stay zero); FW: pairs per batch
template <int Q, int NPROD, int RA, int FW>
__global__ void __launch_bounds__(64 * Q, 2) epic_wide_kernel(FusedParams P) {
  constexpr int NT = 64 * Q, N = 32 * Q, NACC = NPROD == 4 ? 4 : (NPROD == 2 ? 2 : 1), PLW = RA * HS;
  constexpr int NB2 = RA > 32 ? (RA - 32 < 16 ? RA - 32 : 16) : 0, NB3 = RA > 48 ? 16 : 0;
  extern __shared__ __align__(16) unsigned char smem_raw[];
  float4* gh = reinterpret_cast<float4*>(smem_raw);  // [FW][RA][HS]
  float4* tws = gh + FW * PLW;                       // [2Q][TWV]
  float4* E = tws + 2 * Q * TWV;                     // [FW][A]
  uint2* info = reinterpret_cast<uint2*>(E + FW * P.n_ant);  // [R * 32] this channel's cell slots
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  const int n_slot = P.R * S;

  const long long g0 = P.total * (long long)blockIdx.x / gridDim.x;
  const long long g1 = P.total * (long long)(blockIdx.x + 1) / gridDim.x;
  if (g0 >= g1) return;
  constexpr bool TMEM = NPROD == 4;
  constexpr int TCOLS = Q == 4 ? 128 : 64;

  int unit = (int)(g0 / P.nb);
  for (int i = tid; i < n_slot; i += NT) info[i] = __ldg(P.cell_info + (size_t)(unit / Q) * P.cell_stride + i);
  for (int i = tid; i < FW * PLW; i += NT) gh[i] = make_float4(0.0f, 0.0f, 0.0f, 0.0f);
  for (int i = tid; i < 2 * Q * TWV; i += NT) tws[i] = __ldg(P.tw + i);
  __syncthreads();

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

  // S6: as in epic_fused_kernel (direct add when the unit's whole time range ran here, else parked partial sums)
  auto flush = [&](int unit, bool complete, int slot) {
    const int c = unit / Q, l2 = unit - c * Q;
    const size_t plane = (size_t)N * N;
    float* o = P.out + (size_t)c * P.n_planes * plane + (Q * l1 + l2);
    float* part = P.partial + ((size_t)(blockIdx.x * 2 + slot) * NACC * 16) * NT + tid;
    if constexpr (TMEM) {
#pragma unroll
      for (int c4 = 0; c4 < 4; ++c4) {
        float a[16], zero[16];
        tmem_ld16(taddr + 16 * c4, a);
#pragma unroll
        for (int i = 0; i < 16; ++i) zero[i] = 0.0f;
        tmem_st16(taddr + 16 * c4, zero);
#pragma unroll
        for (int kk = 0; kk < 4; ++kk) {
          const int k = 4 * c4 + kk;
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
  int seg_begin = b;
  PrefetchSlots ps;
  prefetch_init<NT, FW>(P, tid, ps);
  uint32_t wlo[MAXW], whi[MAXW];
  prefetch_batch<NT, FW>(P, ps, unit / Q, b, wlo, whi);
  unpack_batch<false>(P, ps, E, wlo, whi, unit / Q);
  __syncthreads();

  const int ntask = FW * P.R * 2;
  for (long long g = g0; g < g1; ++g) {
    int unit_n = unit, b_n = b + 1;
    if (b_n == P.nb) { b_n = 0; ++unit_n; }
    const bool more = g + 1 < g1;
    if (more) prefetch_batch<NT, FW>(P, ps, unit_n / Q, b_n, wlo, whi);

    const int l2 = unit % Q;
    // x-fold constant of the unit: W_Q^{l2} (Q = 4: i^l2, Q = 2: (-1)^l2), exact
    const float fxr = Q == 4 ? (float)((l2 == 0) - (l2 == 2)) : (float)(1 - 2 * l2);
    const float fxi = Q == 4 ? (float)((l2 == 1) - (l2 == 3)) : 0.0f;
    gather_wide<NT, PLW, FW>(P, E, gh, info, n_slot, fxr, fxi);
    __syncthreads();

    for (int base = warp * 32; base < ntask; base += NT) {
      const int task = base + lane;
      const bool valid = task < ntask;
      // idle lanes (only when R < RA) transform the all-zero last row of plane 0
      int f = 0, y = RA - 1, h = 0;
      if (valid) { h = task & 1; const int p = task >> 1; f = p / P.R; y = p - f * P.R; }
      row_task<16>(gh + f * PLW + y * HS, tws + (l2 + Q * h) * TWV, h, valid);
    }
    __syncthreads();

    if (more) unpack_batch<false>(P, ps, E, wlo, whi, unit_n / Q);  // E was last read by this batch's gather
#pragma unroll 1
    for (int f = 0; f < FW; ++f) {
      int tw_off = rho * TWV;
      asm volatile("" : "+r"(tw_off));
      if constexpr (TMEM) col_task_wide_tmem<NB2, NB3>(gh + f * PLW + l1, tws + tw_off, taddr);
      else col_task_wide<NB2, NB3>(gh + f * PLW + l1, tws + tw_off, acc);
    }

    if (unit_n != unit || !more) {
      flush(unit, seg_begin == 0 && b == P.nb - 1, unit == first_unit ? 0 : 1);
      seg_begin = 0;
    }
    if (P.cell_stride != 0 && unit_n / Q != unit / Q && more) {  // per-channel plan: the next channel's cell slots
      for (int i = tid; i < n_slot; i += NT) info[i] = __ldg(P.cell_info + (size_t)(unit_n / Q) * P.cell_stride + i);
    }
    unit = unit_n; b = b_n;
    __syncthreads();  // next batch's E (and cell slots) are complete; gh is free
  }
  if constexpr (TMEM) tmem_free_cta<TCOLS>(tbase, warp);
}

struct WideTables {
  uint2* cell_info;     // [n_layout][R * 32] folded cell slots, sorted by entry count
  float4* tw;           // [2Q][TWV] TwSets with the second fold constant r^32 in word 4
  uint16_t* ent_ant;    // gather entries re-ordered by folded cell: (y, x) entries, then (y, x + 32) entries
  float2* ent_tap;
  int ra;               // rows allocated per plane: 32, 40, 48 or 64
};

template <int Q>
size_t wide_smem_bytes(int ra, int fw, int n_ant_pad, int R) {
  const size_t FW = (size_t)fw;
  return ((size_t)FW * ra * HS + (size_t)2 * Q * TWV + (size_t)FW * n_ant_pad) * sizeof(float4) + (size_t)R * S * sizeof(uint2);
}

template <int Q, int NPROD, int RA, int FW>
int launch_wide(const epic_plan* p, const FusedParams& P, cudaStream_t s) {
  constexpr int NT = 64 * Q, NACC = NPROD == 4 ? 4 : (NPROD == 2 ? 2 : 1);
  const size_t smem = wide_smem_bytes<Q>(RA, FW, P.n_ant, P.R);
  auto kern = epic_wide_kernel<Q, NPROD, RA, FW>;
  if (smem > 48 * 1024)
    EPIC_CUDA_TRY(cudaFuncSetAttribute((const void*)kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
  int per_sm = 0;
  EPIC_CUDA_TRY(cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, kern, NT, smem));
  if (per_sm < 1) return EPIC_ERR_RANGE;
  // kernels that allocate tensor memory: the occupancy query answers 1 although two CTAs share an SM (epic_fused.cu)
  if (NPROD == 4 && 2 * (smem + 1024) <= (size_t)227 * 1024) per_sm = std::max(per_sm, 2);
  const int grid = (int)std::min<long long>(P.total, (long long)per_sm * p->n_sm);
  if ((size_t)grid * 2 * NACC * 16 * NT * sizeof(float) > p->scratch_bytes) return EPIC_ERR_RANGE;
  kern<<<grid, NT, smem, s>>>(P);
  epic_fused_fixup<Q, NPROD><<<(unsigned)(P.total / P.nb), NT, 0, s>>>(P, grid);
  EPIC_CUDA_TRY(cudaGetLastError());
  return EPIC_OK;
}

template <int Q, int NPROD>
int launch_wide_ra(const epic_plan* p, const FusedParams& P, int ra, int fw, cudaStream_t s) {
  if (ra == 32) return launch_wide<Q, NPROD, 32, 4>(p, P, s);
  if (ra == 40) return fw == 3 ? launch_wide<Q, NPROD, 40, 3>(p, P, s) : launch_wide<Q, NPROD, 40, 2>(p, P, s);
  if (ra == 48) return fw == 3 ? launch_wide<Q, NPROD, 48, 3>(p, P, s) : launch_wide<Q, NPROD, 48, 2>(p, P, s);
  return launch_wide<Q, NPROD, 64, 2>(p, P, s);
}

template <int Q>
int launch_wide_q(const epic_plan* p, const FusedParams& P, int n_products, int ra, int fw, cudaStream_t s) {
  if (n_products == 1) return launch_wide_ra<Q, 1>(p, P, ra, fw, s);
  if (n_products == 2) return launch_wide_ra<Q, 2>(p, P, ra, fw, s);
  return launch_wide_ra<Q, 4>(p, P, ra, fw, s);
}

// pairs per batch: as many as keep two CTAs on an SM, and for 48-row planes the count (2 or 3) that leaves
// fewer idle lanes in the row pass (FW * R * 2 tasks on rounds of 64 Q threads)
int wide_fw(int Q, int ra, int R, int n_ant_pad) {
  if (ra == 32) return 4;
  if (ra == 64) return 2;
  const int nt = 64 * Q;
  auto eff = [&](int fw) { const int tasks = fw * R * 2; return (double)tasks / (double)(((tasks + nt - 1) / nt) * nt); };
  const size_t smem3 = Q == 2 ? wide_smem_bytes<2>(ra, 3, n_ant_pad, R) : wide_smem_bytes<4>(ra, 3, n_ant_pad, R);
  if (2 * (smem3 + 1024) > (size_t)227 * 1024) return 2;
  return eff(3) >= eff(2) ? 3 : 2;
}

}  // namespace

// ---------------------------------------------------------------- host side
int wide_plan_init(epic_plan* p) {
  p->wide_ok = 0;
  p->d_wide = nullptr;
  const int Q = p->N / S;
  if (p->N % S != 0 || (Q != 2 && Q != 4)) return EPIC_OK;
  if (p->R > 2 * S || p->Cc > 2 * S) return EPIC_OK;
  if (p->R <= S && p->Cc <= S) return EPIC_OK;  // the 32 x 32 kernel takes it
  if (p->h_ent_ant.size() >= ((size_t)1 << 24)) return EPIC_OK;
  const int R = p->R, ra = R <= 32 ? 32 : (R <= 40 ? 40 : (R <= 48 ? 48 : 64));
  const size_t n_slots = (size_t)R * S;
  std::vector<uint2> info;
  std::vector<uint16_t> ent_ant;
  std::vector<float2> ent_tap;
  ent_ant.reserve(p->h_ent_ant.size());
  ent_tap.reserve(p->h_ent_tap.size());
  for (int l = 0; l < p->n_layout; ++l) {
    // the two cells (y, x') and (y, x' + 32) of every folded slot
    std::vector<const CellRec*> lo(n_slots, nullptr), hi(n_slots, nullptr);
    for (uint32_t i = p->h_cell_off[l]; i < p->h_cell_off[l + 1]; ++i) {
      const CellRec& c = p->h_cells[i];
      if (c.ent_count > 255u) return EPIC_OK;  // falls back to the two-pass path
      (c.x < S ? lo : hi)[(size_t)c.y * S + (c.x % S)] = &c;
    }
    std::vector<uint2> li(n_slots);
    for (size_t s = 0; s < n_slots; ++s) {
      const uint32_t first = (uint32_t)ent_ant.size();
      uint32_t n_lo = 0, n_hi = 0;
      for (int half = 0; half < 2; ++half) {
        const CellRec* c = half ? hi[s] : lo[s];
        if (!c) continue;
        for (uint32_t e = 0; e < c->ent_count; ++e) {
          ent_ant.push_back(p->h_ent_ant[c->ent_begin + e]);
          ent_tap.push_back(p->h_ent_tap[c->ent_begin + e]);
        }
        (half ? n_hi : n_lo) = c->ent_count;
      }
      const uint32_t y = (uint32_t)(s / S), x = (uint32_t)(s % S);
      li[s] = make_uint2((first << 8) | n_lo, (y * HS + x) | (n_hi << 16));
    }
    // sorted by entry count, so that the 32 slots of a warp have (nearly) equal trip counts
    std::stable_sort(li.begin(), li.end(), [](const uint2& a, const uint2& b) {
      return (a.x & 0xFFu) + (a.y >> 16) > (b.x & 0xFFu) + (b.y >> 16);
    });
    info.insert(info.end(), li.begin(), li.end());
  }
  // TwSet of every residue rho = 0..2Q-1 (as fused_plan_init) + r^32 in word 4
  std::vector<float4> tw((size_t)2 * Q * TWV);
  for (int rho = 0; rho < 2 * Q; ++rho) {
    auto cis = [&](double r_pow, int k, int n, float* re, float* im) {  // r^r_pow W_n^k, r = exp(2 pi i rho / N)
      const double ang = 2.0 * M_PI * ((double)rho * r_pow / (double)p->N + (double)k / (double)n);
      *re = (float)std::cos(ang);
      *im = (float)std::sin(ang);
    };
    float v[20] = {0};
    cis(16.0, 0, 1, &v[0], &v[1]);
    cis(8.0, 0, 2, &v[2], &v[3]);
    cis(4.0, 0, 4, &v[4], &v[5]);
    for (int k = 0; k < 2; ++k) cis(2.0, k, 8, &v[6 + 2 * k], &v[7 + 2 * k]);
    for (int k = 0; k < 4; ++k) cis(1.0, k, 16, &v[10 + 2 * k], &v[11 + 2 * k]);
    // r^32 = exp(2 pi i rho / Q): a fourth (or second) root of unity, written exactly
    const int q4 = (rho * 4 / Q) & 3;  // quarter turns
    v[18] = q4 == 0 ? 1.0f : (q4 == 2 ? -1.0f : 0.0f);
    v[19] = q4 == 1 ? 1.0f : (q4 == 3 ? -1.0f : 0.0f);
    for (int j = 0; j < TWV; ++j) tw[(size_t)rho * TWV + j] = make_float4(v[4 * j], v[4 * j + 1], v[4 * j + 2], v[4 * j + 3]);
  }
  WideTables* wt = new (std::nothrow) WideTables();
  if (!wt) return EPIC_ERR_NOMEM;
  wt->cell_info = nullptr; wt->tw = nullptr; wt->ent_ant = nullptr; wt->ent_tap = nullptr;
  wt->ra = ra;
  if (ent_ant.empty()) { ent_ant.push_back(0); ent_tap.push_back(make_float2(0.0f, 0.0f)); }
  cudaError_t ce = cudaMalloc(&wt->cell_info, info.size() * sizeof(uint2));
  if (ce == cudaSuccess) ce = cudaMalloc(&wt->tw, tw.size() * sizeof(float4));
  if (ce == cudaSuccess) ce = cudaMalloc(&wt->ent_ant, ent_ant.size() * sizeof(uint16_t));
  if (ce == cudaSuccess) ce = cudaMalloc(&wt->ent_tap, ent_tap.size() * sizeof(float2));
  if (ce == cudaSuccess) ce = cudaMemcpy(wt->cell_info, info.data(), info.size() * sizeof(uint2), cudaMemcpyHostToDevice);
  if (ce == cudaSuccess) ce = cudaMemcpy(wt->tw, tw.data(), tw.size() * sizeof(float4), cudaMemcpyHostToDevice);
  if (ce == cudaSuccess) ce = cudaMemcpy(wt->ent_ant, ent_ant.data(), ent_ant.size() * sizeof(uint16_t), cudaMemcpyHostToDevice);
  if (ce == cudaSuccess) ce = cudaMemcpy(wt->ent_tap, ent_tap.data(), ent_tap.size() * sizeof(float2), cudaMemcpyHostToDevice);
  p->d_wide = wt;
  if (ce != cudaSuccess) {
    set_cuda_error(ce);
    wide_plan_free(p);
    return ce == cudaErrorMemoryAllocation ? EPIC_ERR_NOMEM : EPIC_ERR_CUDA;
  }
  p->wide_ok = 1;
  return EPIC_OK;
}

void wide_plan_free(epic_plan* p) {
  WideTables* wt = static_cast<WideTables*>(p->d_wide);
  if (wt) {
    if (wt->cell_info) cudaFree(wt->cell_info);
    if (wt->tw) cudaFree(wt->tw);
    if (wt->ent_ant) cudaFree(wt->ent_ant);
    if (wt->ent_tap) cudaFree(wt->ent_tap);
    delete wt;
  }
  p->d_wide = nullptr;
  p->wide_ok = 0;
}

int wide_supported(const epic_plan* p, int is_cf32, int n_pol, int n_products) {
  if (!p->wide_ok || is_cf32) return 0;
  if (!((n_pol == 1 && n_products == 1) || (n_pol == 2 && (n_products == 2 || n_products == 4)))) return 0;
  const WideTables* wt = static_cast<const WideTables*>(p->d_wide);
  const int Q = p->N / S, nt = 64 * Q, a_pad = (p->n_ant + 3) & ~3;
  const int fw = wide_fw(Q, wt->ra, p->R, a_pad);
  if ((long long)fw * (a_pad / 4) > (long long)MAXW * nt) return 0;  // prefetch registers
  const size_t smem = Q == 2 ? wide_smem_bytes<2>(wt->ra, fw, a_pad, p->R) : wide_smem_bytes<4>(wt->ra, fw, a_pad, p->R);
  return smem <= (size_t)200 * 1024 ? 1 : 0;
}

int wide_image(epic_plan* p, const ImageArgs& a) {
  const WideTables* wt = static_cast<const WideTables*>(p->d_wide);
  const int Q = p->N / S;
  FusedParams P;
  P.volt = static_cast<const uint8_t*>(a.volt);
  P.out = a.out;
  P.cell_info = wt->cell_info;
  P.cell_stride = p->n_layout > 1 ? p->R * S : 0;
  P.ent_ant = wt->ent_ant;
  P.ent_tap = wt->ent_tap;
  P.tw = wt->tw;
  P.partial = static_cast<float*>(p->d_scratch);
  P.native = a.native;
  P.phasor = a.phasor_pair;
  P.n_t = a.n_t;
  P.n_chan = a.n_chan;
  P.n_ant = (p->n_ant + 3) & ~3;
  P.n_ant_true = p->n_ant;
  P.unaligned = (p->n_ant & 3) != 0 || (reinterpret_cast<uintptr_t>(a.volt) & 3u) != 0;  // then the prefetch reads bytes
  P.n_ent = p->t.n_ent;
  P.n_pol = a.n_pol;
  P.n_planes = a.n_planes;
  P.R = p->R;
  P.Cc = p->Cc;
  const int fw = wide_fw(Q, wt->ra, p->R, P.n_ant);
  const int per_batch = a.n_pol == 2 ? fw : 2 * fw;  // time samples per batch
  P.pairs_per_batch = fw;
  P.nb = (a.n_t + per_batch - 1) / per_batch;
  P.total = (long long)a.n_chan * Q * P.nb;
  const int st = Q == 2 ? launch_wide_q<2>(p, P, a.n_products, wt->ra, fw, a.stream) : launch_wide_q<4>(p, P, a.n_products, wt->ra, fw, a.stream);
  if (st != EPIC_OK) return st;
  p->last_launches = 2;  // the wide kernel and the (tiny) fix-up of split units
  return EPIC_OK;
}

}  // namespace epic
