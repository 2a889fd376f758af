// Tiled two-pass EPIC path for large planes (N = 256, 512; any support): the packed (f32x2)
// transform core of epic_packed.cuh, with the row-transformed plane H passed between two kernels
// through the plan's scratch (BASELINE.json north_star (3): a two-pass FFT only when the grid
// exceeds shared memory; the scratch is 1 GiB by default, epic_plan_set_scratch_limit caps a
// batch so that H stays resident in the 126 MB L2).  PAPER.md:122-126 steps S1..S6.
//
//   kernel A  tiled_rows   S1 unpack the frame's voltages -> E (shared), S3 gather-gridding of a
//                          group of occupied rows, S4 along x -> H[frame][y][l] (float4 pairs)
//   kernel B  tiled_cols   S4 along y for a strip of W image columns, S5 products, S6
//                          accumulation over the batch's time samples in registers, one add into
//                          out_accum per batch (the CTA is the only writer of its pixels)
//
// Pruning.  Only the R x Cc box of occupied cells exists (relocated to the origin, Q7).
// An N-point transform of a sequence whose elements y >= N/2 are (almost all) zero is two
// half-transforms, outputs 2k + rho, rho = 0, 1:
//
//   X[2k + rho] = sum_{y < M} s_rho[y] r^y W_M^{y k},  M = N/2, r = W_N^{rho},
//   s_rho[y] = in[y] + (-1)^rho in[y + M]   (only y < nb = R - M has a partner: the "prefold")
//
// Each half-transform of length M = 16 J (J = 8, 16) is done by a team of J threads:
//   step 1  thread j: 16-point ramped FFT of s[J i + j], base r^J           -> U_j[k1]
//   step 2  thread t: J-point ramped FFT over j of U_j[k1], base r W_M^{k1} -> X[k1 + 16 k2]
// with the two steps exchanging through shared memory.  The ramps are absorbed into the butterfly
// twiddles (epic_packed.cuh), which come from plan tables computed in double.
#include <algorithm>
#include <cmath>
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <new>
#include <vector>

#include "epic_internal.h"
#include "epic_packed.cuh"

namespace epic {
namespace {

// threads of tiled_rows: small CTAs, so that several row groups are in flight per SM and one CTA's
// gather latency (dependent L2 reads between two barriers) overlaps the other CTAs' transforms:
// measured on C4 256 / 128 / 64 threads -> 2.39 / 2.58 / 2.68 M frames/s, on C5 0.463 / 0.483 / 0.461
template <int J> constexpr int NT_A = (J == 8) ? 64 : 128;
constexpr int NT_B = 128;  // threads of tiled_cols
constexpr int XJ = 17;     // exchange buffer: [team][j][XJ] float4, k1 < 16 (padded: conflict-free both ways)

template <int J> constexpr int x_team_stride() { return ((J * XJ + 7) / 8) * 8 + 4; }  // = 4 mod 8
// tiled_cols: a quarter-warp is 8 teams with one j, so consecutive teams must fall in distinct bank groups
template <int J> constexpr int x_team_stride_cols() { return (J * XJ) | 1; }
constexpr int bitrev3(int v) { return ((v & 1) << 2) | (v & 2) | ((v & 4) >> 2); }
constexpr int bitrev4t(int v) { return ((v & 1) << 3) | ((v & 2) << 1) | ((v & 4) >> 1) | ((v & 8) >> 3); }

struct TiledParams {
  DevTables t;
  const uint8_t* volt;   // [T][C][Np][A]
  float4* H;             // scratch [frame][R][N]
  float* out;            // [C][planes][N][N]
  const float4* tw1;     // [2][TWV]      step-1 TwSet of rho (base r^J)
  const float4* tw2;     // [2][16][TWV]  step-2 twiddles of (rho, k1) (base r W_M^{k1})
  const float4* ent_rec; // [n_ent] gather entries as one 16-byte record: (tap.re, tap.im, antenna index bits, 0)
  int n_t, n_chan, n_pol, n_planes;
  int c0, p0, Cb, Tb;    // batch: channels [c0, c0+Cb) x pairs [p0, p0+Tb)
  int nbx, nby;          // prefold counts along x (row pass) and y (column pass)
  int native;            // input order [T][C][A][Np] instead of [T][C][Np][A]
  const float4* phasor;  // delay phasors, pair-packed [C][A], or nullptr
};

__device__ __forceinline__ void cp_async16(void* smem_dst, const void* gmem_src) {
  const unsigned d = (unsigned)__cvta_generic_to_shared(smem_dst);
  asm volatile("cp.async.cg.shared.global [%0], [%1], 16;" ::"r"(d), "l"(gmem_src) : "memory");
}
__device__ __forceinline__ void cp_async_commit() { asm volatile("cp.async.commit_group;" ::: "memory"); }
__device__ __forceinline__ void cp_async_wait_all() { asm volatile("cp.async.wait_group 0;" ::: "memory"); }

__device__ __forceinline__ C2 to_c2(float4 v) { return C2{make_float2(v.x, v.y), make_float2(v.z, v.w)}; }
__device__ __forceinline__ float4 to_f4(const C2& z) { return make_float4(z.re.x, z.re.y, z.im.x, z.im.y); }

// ---------------------------------------------------------------- kernel A: unpack, grid, row transforms
// Work item = (frame pair of the batch, group of RG occupied rows); every CTA takes an equal contiguous
// range of items (one wave, no tail) and re-unpacks E when its frame changes.
// Thread roles in the transform steps: tid = rho + 2 j + 2 J r  (row r of the group, team (r, rho)).
// One shared buffer BUF serves in turn as the gridded rows RB[RG][N], the exchange buffer
// X[team][j][XJ] and the transformed rows; registers carry the data across the hand-overs.
template <int J, bool DELTA>
__global__ void __launch_bounds__(NT_A<J>) tiled_rows(TiledParams P) {
  constexpr int N = 32 * J, M = 16 * J, RG = NT_A<J> / (2 * J), XS = x_team_stride<J>();
  constexpr int BUF = (RG * N > 2 * RG * XS) ? RG * N : 2 * RG * XS;
  extern __shared__ __align__(16) unsigned char smem_raw[];
  float4* buf = reinterpret_cast<float4*>(smem_raw);  // [BUF]
  float4* tw1 = buf + BUF;                            // [2][TWV]
  float4* tw2 = tw1 + 2 * TWV;                        // [2][16][TWV]
  uint32_t* E = reinterpret_cast<uint32_t*>(tw2 + 2 * 16 * TWV);  // [A] biased bytes (epic_packed.cuh)
  const int tid = threadIdx.x;
  const DevTables& t = P.t;
  for (int i = tid; i < 2 * TWV; i += NT_A<J>) tw1[i] = __ldg(P.tw1 + i);
  for (int i = tid; i < 2 * 16 * TWV; i += NT_A<J>) tw2[i] = __ldg(P.tw2 + i);

  const int rho = tid & 1, j = (tid >> 1) & (J - 1), r = tid / (2 * J);
  float4* xt = buf + (2 * r + rho) * XS;  // this team's exchange block
  const int n_groups = (t.R + RG - 1) / RG;
  const long long n_items = (long long)P.Cb * P.Tb * n_groups;
  const int item0 = (int)(n_items * blockIdx.x / gridDim.x), item1 = (int)(n_items * (blockIdx.x + 1) / gridDim.x);
  int fb_loaded = -1;
  const float4* ph_c = nullptr;  // this frame's channel's delay phasors
  for (int i = tid; i < RG * N; i += NT_A<J>) buf[i] = make_float4(0.0f, 0.0f, 0.0f, 0.0f);
  for (int item = item0; item < item1; ++item) {
    const int fb = item / n_groups, g = item - fb * n_groups;
    if (fb != fb_loaded) {  // S1: this frame pair's voltages -> E
      fb_loaded = fb;
      const int cb = fb / P.Tb, pb = fb - cb * P.Tb;
      const int c = P.c0 + cb, pair = P.p0 + pb;
      const int t_lo = P.n_pol == 2 ? pair : 2 * pair, t_hi = P.n_pol == 2 ? pair : 2 * pair + 1;
      const size_t row_bytes = (size_t)P.n_pol * t.n_ant;
      const uint8_t* lo = P.volt + ((size_t)t_lo * P.n_chan + c) * row_bytes;
      const uint8_t* hi = P.volt + ((size_t)t_hi * P.n_chan + c) * row_bytes + (P.n_pol == 2 ? t.n_ant : 0);
      for (int q = tid; q < (t.n_ant >> 2); q += NT_A<J>) {
        uint32_t wlo = 0u, whi = 0u;
        if (P.native && P.n_pol == 2) {  // (a X, a Y) byte pairs
          if (t_lo < P.n_t) deinterleave_pols(__ldg(reinterpret_cast<const uint32_t*>(lo) + 2 * q),
                                              __ldg(reinterpret_cast<const uint32_t*>(lo) + 2 * q + 1), wlo, whi);
        } else {
          if (t_lo < P.n_t) wlo = __ldg(reinterpret_cast<const uint32_t*>(lo) + q);
          if (t_hi < P.n_t) whi = __ldg(reinterpret_cast<const uint32_t*>(hi) + q);
        }
        *reinterpret_cast<uint4*>(E + 4 * q) = unpack_words_b8(wlo, whi);
      }
      ph_c = P.phasor ? P.phasor + (size_t)c * t.n_ant : nullptr;
    }
    __syncthreads();  // E and the zeroed row buffer (end of the previous item) are complete
    const int y0 = g * RG, rows = min(RG, t.R - y0);
    // S3: gather-gridding of the group's cells, one thread per cell, sums in table order.
    // Four cell records, then four entry records, are in flight per thread (L2 latency).
    const uint32_t* rp = t.row_ptr + (size_t)(P.c0 + fb / P.Tb) * t.row_stride;  // this channel's layout
    const uint32_t cbeg = __ldg(rp + y0), cend = __ldg(rp + y0 + rows);
    for (uint32_t base = cbeg + tid; base < cend; base += 4 * NT_A<J>) {
      CellRec cr[4];
#pragma unroll
      for (int q = 0; q < 4; ++q) cr[q] = t.cells[min(base + q * NT_A<J>, cend - 1)];
#pragma unroll
      for (int q = 0; q < 4; ++q) {
        if (base + q * NT_A<J> >= cend) break;
        const CellRec cell = cr[q];
        float2 sr = make_float2(0.0f, 0.0f), si = make_float2(0.0f, 0.0f);
        const uint32_t e_end = cell.ent_begin + cell.ent_count;
        for (uint32_t e = cell.ent_begin; e < e_end; e += 4) {
          float4 rec[4];  // (tap.re, tap.im, antenna, -)
#pragma unroll
          for (int k = 0; k < 4; ++k) rec[k] = __ldg(P.ent_rec + min(e + k, e_end - 1));
#pragma unroll
          for (int k = 0; k < 4; ++k) {
            if (e + k < e_end) {
              float2 vr, vi;
              const uint32_t ant = __float_as_uint(rec[k].z);
              b8_to_pair(E[ant], vr, vi);
              if (ph_c) {  // delay compensation (reading Q19)
                const float4 pp = __ldg(ph_c + ant);
                const float2 pr = make_float2(pp.x, pp.y), pi = make_float2(pp.z, pp.w);
                const float2 r2 = __ffma2_rn(vr, pr, neg2(__fmul2_rn(vi, pi)));
                vi = __ffma2_rn(vr, pi, __fmul2_rn(vi, pr));
                vr = r2;
              }
              if (DELTA) {
                sr = __fadd2_rn(sr, vr); si = __fadd2_rn(si, vi);
              } else {
                sr = __ffma2_rn(vr, f2(rec[k].x), sr); sr = __ffma2_rn(neg2(vi), f2(rec[k].y), sr);
                si = __ffma2_rn(vi, f2(rec[k].x), si); si = __ffma2_rn(vr, f2(rec[k].y), si);
              }
            }
          }
        }
        buf[(cell.y - y0) * N + cell.x] = make_float4(sr.x, sr.y, si.x, si.y);
      }
    }
    __syncthreads();
    C2 z[16];
    {  // step 1 inputs: s_rho[J i + j] = in[x] +- in[x + M] for the nbx elements that have a partner
      const float4* row = buf + r * N;
#pragma unroll
      for (int i = 0; i < 16; ++i) {
        const int x = J * i + j;
        C2 a = to_c2(row[x]);
        if (x < P.nbx) {
          const C2 b = to_c2(row[x + M]);
          const float2 sg = f2(rho ? -1.0f : 1.0f);
          a.re = __ffma2_rn(b.re, sg, a.re); a.im = __ffma2_rn(b.im, sg, a.im);
        }
        z[bitrev4t(i)] = a;
      }
    }
    __syncthreads();  // every thread holds its inputs: buf becomes the exchange buffer
    {
      const float4* tw = tw1 + rho * TWV;
      const float4 t0 = tw[0];
      fft16_ramped(z, tw, t0.z, t0.w);
#pragma unroll
      for (int k1 = 0; k1 < 16; ++k1) xt[j * XJ + k1] = to_f4(z[k1]);
    }
    __syncthreads();
    // step 2: thread t = j takes k1 = t (and t + 8 when J == 8); outputs l = 2 (k1 + 16 k2) + rho go
    // straight to H: for one k2 the 2 J lanes of a team write 2 J consecutive float4
    float4* hrow = P.H + ((size_t)fb * t.R + y0 + r) * N + rho;
    if constexpr (J == 8) {
      C2 za[8], zb[8];
#pragma unroll
      for (int q = 0; q < 8; ++q) { za[bitrev3(q)] = to_c2(xt[q * XJ + j]); zb[bitrev3(q)] = to_c2(xt[q * XJ + j + 8]); }
      __syncthreads();  // exchange buffer consumed: the row buffer is zeroed for the next item
      for (int i = tid; i < RG * N; i += NT_A<J>) buf[i] = make_float4(0.0f, 0.0f, 0.0f, 0.0f);
      const float4 *ta = tw2 + (rho * 16 + j) * TWV, *tb = tw2 + (rho * 16 + j + 8) * TWV;
      const float4 a0 = ta[0], a1 = ta[1], b0 = tb[0], b1 = tb[1];
      fft8_ramped(za, a0.x, a0.y, a0.z, a0.w, a1.x, a1.y, a1.z, a1.w);
      fft8_ramped(zb, b0.x, b0.y, b0.z, b0.w, b1.x, b1.y, b1.z, b1.w);
      if (r < rows) {
#pragma unroll
        for (int k2 = 0; k2 < 8; ++k2) {
          hrow[2 * (j + 16 * k2)] = to_f4(za[k2]);
          hrow[2 * (j + 8 + 16 * k2)] = to_f4(zb[k2]);
        }
      }
    } else {
#pragma unroll
      for (int q = 0; q < 16; ++q) z[bitrev4t(q)] = to_c2(xt[q * XJ + j]);
      __syncthreads();
      for (int i = tid; i < RG * N; i += NT_A<J>) buf[i] = make_float4(0.0f, 0.0f, 0.0f, 0.0f);
      const float4* tw = tw2 + (rho * 16 + j) * TWV;
      const float4 t0 = tw[0];
      fft16_ramped(z, tw, t0.z, t0.w);
      if (r < rows) {
#pragma unroll
        for (int k2 = 0; k2 < 16; ++k2) hrow[2 * (j + 16 * k2)] = to_f4(z[k2]);
      }
    }
  }
}

// ---------------------------------------------------------------- kernel B: column transforms, products, accumulation
// CTA = (strip of W = 64/J image columns, channel of the batch); it loops over the batch's Tb frame
// pairs with the accumulators of its W x N pixels in registers and adds them into out_accum once.
// Thread roles: tid = rho + 2 w + 2 W j (column w of the strip, team (w, rho)): the two residues of a
// column sit in adjacent lanes (merged LDS.128), a half-warp reads whole 128-byte tile rows.
template <int NPROD>
__device__ __forceinline__ void accumulate_products(const C2& z, float2& acc, float2& xy) {
  acc = __ffma2_rn(z.re, z.re, acc);
  acc = __ffma2_rn(z.im, z.im, acc);
  if constexpr (NPROD == 4) {  // XY = A_lo conj(A_hi) (reading Q11)
    xy.x = fmaf(z.re.x, z.re.y, xy.x); xy.x = fmaf(z.im.x, z.im.y, xy.x);
    xy.y = fmaf(z.im.x, z.re.y, xy.y); xy.y = fmaf(-z.re.x, z.im.y, xy.y);
  }
}

template <int J, int NPROD>
__global__ void __launch_bounds__(NT_B, 3) tiled_cols(TiledParams P) {
  constexpr int N = 32 * J, M = 16 * J, W = 64 / J, XS = x_team_stride_cols<J>();
  extern __shared__ __align__(16) unsigned char smem_raw[];
  const DevTables& t = P.t;
  const int R = t.R;
  float4* xbuf = reinterpret_cast<float4*>(smem_raw);  // [2W][XS]
  float4* tw1 = xbuf + 2 * W * XS;                     // [2][TWV]
  float4* tw2 = tw1 + 2 * TWV;                         // [2][16][TWV]
  float4* tile = tw2 + 2 * 16 * TWV;                   // [2][R + 1][W]; row R stays zero
  const int tile_sz = (R + 1) * W;
  const int tid = threadIdx.x;
  const int rho = tid & 1, w = (tid >> 1) & (W - 1), j = tid / (2 * W);
  const int l0 = blockIdx.x * W, cb = blockIdx.y, c = P.c0 + cb;
  float4* xt = xbuf + (2 * w + rho) * XS;

  for (int i = tid; i < 2 * TWV; i += NT_B) tw1[i] = __ldg(P.tw1 + i);
  for (int i = tid; i < 2 * 16 * TWV; i += NT_B) tw2[i] = __ldg(P.tw2 + i);
  if (tid < 2 * W) tile[(tid / W) * tile_sz + R * W + (tid % W)] = make_float4(0.0f, 0.0f, 0.0f, 0.0f);

  auto stage = [&](int pb, int b) {  // H[frame][y][l0 .. l0+W) -> tile[b], 16 bytes per copy
    const float4* src = P.H + ((size_t)(cb * P.Tb + pb) * R) * N + l0;
    float4* dst = tile + b * tile_sz;
    for (int i = tid; i < R * W; i += NT_B) {
      const int y = i / W, ww = i - y * W;
      cp_async16(dst + i, src + (size_t)y * N + ww);
    }
    cp_async_commit();
  };

  float2 acc[16], xy[NPROD == 4 ? 16 : 1];
#pragma unroll
  for (int k = 0; k < 16; ++k) acc[k] = make_float2(0.0f, 0.0f);
#pragma unroll
  for (int k = 0; k < (NPROD == 4 ? 16 : 1); ++k) xy[k] = make_float2(0.0f, 0.0f);

  stage(0, 0);
  for (int pb = 0; pb < P.Tb; ++pb) {
    float4* cur = tile + (pb & 1) * tile_sz;
    cp_async_wait_all();
    __syncthreads();  // this frame's tile is complete; the previous frame is done with xbuf and the other tile
    if (pb + 1 < P.Tb) stage(pb + 1, (pb + 1) & 1);
    {  // step 1
      C2 z[16];
#pragma unroll
      for (int i = 0; i < 16; ++i) {
        const int y = J * i + j;
        const int ys = y < R ? y : R;  // rows beyond the occupied box: the zero row
        C2 a = to_c2(cur[ys * W + w]);
        if (y < P.nby) {  // the few rows that have a partner y + M (prefold)
          const C2 b = to_c2(cur[(y + M) * W + w]);
          const float2 sg = f2(rho ? -1.0f : 1.0f);
          a.re = __ffma2_rn(b.re, sg, a.re); a.im = __ffma2_rn(b.im, sg, a.im);
        }
        z[bitrev4t(i)] = a;
      }
      const float4* tw = tw1 + rho * TWV;
      const float4 t0 = tw[0];
      fft16_ramped(z, tw, t0.z, t0.w);
#pragma unroll
      for (int k1 = 0; k1 < 16; ++k1) xt[j * XJ + k1] = to_f4(z[k1]);
    }
    __syncthreads();
    if constexpr (J == 8) {  // step 2 + S5 + S6: k1 = j and j + 8
#pragma unroll
      for (int half = 0; half < 2; ++half) {
        C2 z[8];
        const int k1 = j + 8 * half;
#pragma unroll
        for (int q = 0; q < 8; ++q) z[bitrev3(q)] = to_c2(xt[q * XJ + k1]);
        const float4* tw = tw2 + (rho * 16 + k1) * TWV;
        const float4 a0 = tw[0], a1 = tw[1];
        fft8_ramped(z, a0.x, a0.y, a0.z, a0.w, a1.x, a1.y, a1.z, a1.w);
#pragma unroll
        for (int k2 = 0; k2 < 8; ++k2) accumulate_products<NPROD>(z[k2], acc[8 * half + k2], xy[NPROD == 4 ? 8 * half + k2 : 0]);
      }
    } else {
      C2 z[16];
#pragma unroll
      for (int q = 0; q < 16; ++q) z[bitrev4t(q)] = to_c2(xt[q * XJ + j]);
      const float4* tw = tw2 + (rho * 16 + j) * TWV;
      const float4 t0 = tw[0];
      fft16_ramped(z, tw, t0.z, t0.w);
#pragma unroll
      for (int k2 = 0; k2 < 16; ++k2) accumulate_products<NPROD>(z[k2], acc[k2], xy[NPROD == 4 ? k2 : 0]);
    }
  }
  // S6: one add per pixel; this CTA is the only writer of (channel c, columns l0 .. l0+W)
  const size_t plane = (size_t)N * N;
  float* o = P.out + (size_t)c * P.n_planes * plane + (l0 + w);
#pragma unroll
  for (int i = 0; i < 16; ++i) {
    const int k1 = (J == 8) ? j + 8 * (i >> 3) : j, k2 = (J == 8) ? (i & 7) : i;
    float* px = o + (size_t)(2 * (k1 + 16 * k2) + rho) * N;
    if constexpr (NPROD == 1) {
      px[0] += acc[i].x + acc[i].y;
    } else {
      px[0] += acc[i].x;
      px[plane] += acc[i].y;
    }
    if constexpr (NPROD == 4) {  // YX = conj(XY)
      px[2 * plane] += xy[i].x;
      px[3 * plane] += xy[i].y;
      px[4 * plane] += xy[i].x;
      px[5 * plane] -= xy[i].y;
    }
  }
}

// ================================================================ streamed variant (EPIC_PATH_STREAM)
// The same two transform passes as ONE persistent, cooperatively launched kernel with two CTA roles,
// so that the row-transformed plane H never goes to HBM and out_accum is touched once per call
// (BASELINE.json north_star (3), (4); PAPER.md:223 is the memory-bound regime this avoids):
//
//   row CTAs   (producers)  one per (channel of the wave, group of RG occupied rows).  The group's
//              gather tables (taps, antenna indices, per-cell entry ranges) are built in shared memory
//              once per wave; per time sample the CTA fetches only the voltage BYTES its entries need
//              (prefetched one sample ahead, no whole-frame unpack), grids, transforms its rows and
//              writes them into slot (s mod Tring) of the channel's ring in the plan's scratch.
//   column CTAs (consumers) one per (channel of the wave, strip of W image columns), as tiled_cols, but
//              looping over ALL time samples of the call with the accumulators in registers; one add
//              into out_accum per channel.
//
// A wave is Cw channels (as many as fit the resident CTA slots); the kernel loops over the waves.
// Hand-over per (channel slot cl, frame sequence number s = wave * n_pairs + pair): ready[cl][s]
// counts the row CTAs that have written their rows of frame s (release), consumed[cl][s] the column
// CTAs that have copied their tile of it into shared memory; a producer reuses a ring slot only
// after consumed[cl][s - Tring] == strips.  The ring is sized to stay resident in the 126 MB L2.
// All CTAs are co-resident (cooperative launch), so the waits cannot deadlock; a wait that
// exceeds ~4 s traps instead of hanging the device.
constexpr int NT_S = 128;     // threads of either role
constexpr int PF_MAX = 16;    // prefetched entries per row-CTA thread: a row group holds <= PF_MAX * NT_S gather entries

struct StreamParams {
  TiledParams b;
  int* flags;          // [Cw][n_seq][2] = (ready, consumed) per hand-over block, zeroed before every call; n_seq = n_waves * nbw
  int Cw, n_waves, n_pairs, n_seq, Tring, n_groups, strips;
  int B, nbw, TB;      // hand-over block: B frames; blocks per wave; ring length in blocks (Tring = TB * B frames)
  int K;               // row CTAs per (channel, row group), interleaved in time: CTA k takes the pairs p = k mod K
  int ent_cap;         // gather entries a row CTA's shared tables can hold
  unsigned long long* stats;  // development: [0] column-role wait cycles, [1] row-role wait cycles, [2], [3] their total cycles
};

__device__ __forceinline__ int ld_acquire_gpu(const int* p) {
  int v;
  asm volatile("ld.acquire.gpu.global.s32 %0, [%1];" : "=r"(v) : "l"(p) : "memory");
  return v;
}
__device__ __forceinline__ void red_release_gpu_add(int* p, int v) {
  asm volatile("red.release.gpu.global.add.s32 [%0], %1;" ::"l"(p), "r"(v) : "memory");
}
// one thread: spin until *flag >= target (bounded: a lost hand-over traps instead of hanging the GPU)
__device__ __forceinline__ void wait_flag_ge(const int* flag, int target, unsigned long long* stat = nullptr) {
  const long long t00 = stat ? clock64() : 0;
  struct Acc { unsigned long long* s; long long t; __device__ ~Acc() { if (s) atomicAdd(s, (unsigned long long)(clock64() - t)); } } acc{stat, t00};
  if (ld_acquire_gpu(flag) >= target) return;
  const long long t0 = clock64();
  while (ld_acquire_gpu(flag) < target) {
    __nanosleep(64);
    if (clock64() - t0 > (8LL << 30)) __trap();
  }
}

// stage word of one gather entry: (lo byte, hi byte) = the 4+4-bit samples of its antenna in the two
// planes of the pair (pol X / pol Y, or two consecutive time samples); S1 happens at use.
__device__ __forceinline__ void stage_to_pair(uint32_t x, float2& vr, float2& vi) {
  // bytes (re_lo+8, re_hi+8, im_lo+8, im_hi+8), as unpack_words_b8 makes them (epic_packed.cuh)
  const uint32_t w = (((x >> 4) & 0x0F0Fu) | ((x & 0x0F0Fu) << 16)) ^ 0x08080808u;
  b8_to_pair(w, vr, vi);
}

template <int J> constexpr int stream_rg() { return NT_S / (2 * J); }
// bytes per gather entry in a row CTA's shared tables: tap (MODE 1: float2, MODE 2: float4 tap x phasor
// of both planes), antenna index, two stage words
template <int MODE> constexpr int stream_ent_bytes() { return (MODE == 0 ? 0 : (MODE == 1 ? 8 : 16)) + 2 + 4; }

// Thread roles of both stream roles: the J threads of a transform team, and the two teams (rho = 0, 1) of
// one row / column, sit in ONE warp -- lane = rho + 2 j + 2 J b, item = warp * (16 / J) + b -- so the
// step-1 / step-2 exchange through shared memory needs only __syncwarp(), not a CTA barrier (the first
// version of this kernel had 6 CTA barriers per row item: `barrier` was 6.3 of its 12 stall cycles per
// issue, profiles/r02_large_grid_ncu.md).  The two residues of a row / column are in adjacent lanes
// (LDS.128 merges same-address lane pairs).
// Exchange block of a team: [J][16] float4, element (j, k1) at j * 16 + (k1 ^ j ^ 4 rho): the XOR
// swizzle keeps a quarter-warp's 8 accesses in 8 distinct 16-byte bank groups both ways, unpadded.
__device__ __forceinline__ int xsw(int j, int k1, int rho) { return j * 16 + ((k1 ^ j ^ (rho << 2)) & 15); }

// ---- producer role: S1 + S3 + S4 along x for (channel slot cl, row group g, time phase kph of K),
// every wave.  MODE 0: delta kernel (sums of samples); 1: complex taps; 2: taps times the channel's
// delay phasors.
template <int J, int MODE>
__device__ __forceinline__ void stream_rows_role(const StreamParams& S, float4* tw1, float4* tw2, unsigned char* smem,
                                                 int cl, int g, int kph) {
  constexpr int N = 32 * J, M = 16 * J, RG = stream_rg<J>();
  const TiledParams& P = S.b;
  const DevTables& t = P.t;
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5, cap = S.ent_cap;
  float4* buf = reinterpret_cast<float4*>(smem);                       // [RG][N] gridded rows; a row's region is
                                                                       // also its two teams' exchange blocks
  unsigned char* q = smem + (size_t)RG * N * sizeof(float4);
  float2* tab2 = reinterpret_cast<float2*>(q);                         // MODE 1: [cap] taps
  float4* tab4 = reinterpret_cast<float4*>(q);                         // MODE 2: [cap] (tr_lo, tr_hi, ti_lo, ti_hi)
  q += (size_t)cap * (MODE == 0 ? 0 : (MODE == 1 ? 8 : 16));
  uint16_t* ant = reinterpret_cast<uint16_t*>(q);                      // [cap]
  uint16_t* stage = ant + cap;                                         // [2][cap]
  uint32_t* crec = reinterpret_cast<uint32_t*>(stage + 2 * cap);       // [n_cell] nonempty cells of the group:
                                                                       // offset in buf (11 bits) | first entry (12) | entries (9)
  const int rho = lane & 1, j = (lane >> 1) & (J - 1), r = warp * (16 / J) + lane / (2 * J);
  float4* row = buf + r * N;
  float4* xt = row + rho * (J * 16);
  const int y0 = g * RG, rows = min(RG, t.R - y0);
  int ncell = 0;
  const size_t row_bytes = (size_t)P.n_pol * t.n_ant;
  int n_e = 0, next_sig = 0, waited = -1;  // hand-over state: first block not yet announced / last block waited for
  for (int i = tid; i < RG * N; i += NT_S) buf[i] = make_float4(0.0f, 0.0f, 0.0f, 0.0f);

  for (int w = 0; w < S.n_waves; ++w) {
    const int c = w * S.Cw + cl;
    if (c >= P.n_chan) break;
    if (w == 0 || t.n_layout > 1 || MODE == 2) {  // the group's gather tables (per layout / per channel's phasors)
      __syncthreads();
      const uint32_t* rp = t.row_ptr + (size_t)c * t.row_stride;
      const uint32_t cbeg = __ldg(rp + y0), cend = __ldg(rp + y0 + rows);
      uint32_t e0 = 0;
      n_e = 0;
      if (cbeg < cend) {
        const CellRec last = t.cells[cend - 1];
        e0 = t.cells[cbeg].ent_begin;
        n_e = (int)(last.ent_begin + last.ent_count - e0);
      }
      ncell = (int)(cend - cbeg);
      for (uint32_t i = cbeg + tid; i < cend; i += NT_S) {
        const CellRec cell = t.cells[i];
        crec[i - cbeg] = (uint32_t)((cell.y - y0) * N + cell.x) | ((cell.ent_begin - e0) << 11) | (cell.ent_count << 23);
      }
      for (int e = tid; e < n_e; e += NT_S) {
        const uint32_t a = __ldg(t.ent_ant + e0 + e);
        ant[e] = (uint16_t)a;
        if constexpr (MODE != 0) {
          const float2 wv = __ldg(t.ent_tap + e0 + e);
          if constexpr (MODE == 1) {
            tab2[e] = wv;
          } else {  // delay compensation (reading Q19) folded into the tap, per plane of the pair
            const float4 pp = __ldg(P.phasor + (size_t)c * t.n_ant + a);  // (re_lo, re_hi, im_lo, im_hi)
            tab4[e] = make_float4(wv.x * pp.x - wv.y * pp.z, wv.x * pp.y - wv.y * pp.w,
                                  wv.x * pp.z + wv.y * pp.x, wv.x * pp.w + wv.y * pp.y);
          }
        }
      }
    }
    // S1 input: the bytes of this group's entries for one pair (PAPER.md:120 input orders)
    // The two bytes of an entry stay in separate registers until put(): combining them at the load would make every
    // load wait for its data there (measured: 15 % of the row role's stall samples were this one line; C5 +32 %)
    uint32_t pf[PF_MAX], pg[PF_MAX];
    auto fetch = [&](int pair) {
      const int t_lo = P.n_pol == 2 ? pair : 2 * pair, t_hi = P.n_pol == 2 ? pair : 2 * pair + 1;
      const uint8_t* lo = P.volt + ((size_t)t_lo * P.n_chan + c) * row_bytes;
      const uint8_t* hi = P.volt + ((size_t)t_hi * P.n_chan + c) * row_bytes + (P.n_pol == 2 ? t.n_ant : 0);
      const bool have_hi = t_hi < P.n_t;
#pragma unroll
      for (int k = 0; k < PF_MAX; ++k) {
        const int e = tid + k * NT_S;
        pf[k] = 0u; pg[k] = 0u;
        if (e < n_e) {
          const uint32_t a = ant[e];
          if (P.native && P.n_pol == 2) {
            pf[k] = __ldg(lo + 2 * a);          // (a X, a Y) adjacent bytes, fetched one by one: any pointer alignment
            pg[k] = __ldg(lo + 2 * a + 1);
          } else {
            pf[k] = __ldg(lo + a);
            if (have_hi) pg[k] = __ldg(hi + a);
          }
        }
      }
    };
    auto put = [&](int b) {
#pragma unroll
      for (int k = 0; k < PF_MAX; ++k) {
        const int e = tid + k * NT_S;
        if (e < n_e) stage[b * cap + e] = (uint16_t)(pf[k] | (pg[k] << 8));
      }
    };
    __syncthreads();  // ant[] and crec[] are complete
    int cur = 0;
    if (kph < S.n_pairs) { fetch(kph); put(0); }
    // ring slot of frame p: (block gb mod TB) * B + p mod B, kept incrementally (no divisions in the loop)
    int pb = kph / S.B, pr = kph - pb * S.B, rb = (w * S.nbw + pb) % S.TB;
    for (int p = kph; p < S.n_pairs; p += S.K) {
      const int gb = w * S.nbw + pb, slot = rb * S.B + pr;  // hand-over block and ring slot of this frame
      if (p + S.K < S.n_pairs) fetch(p + S.K);
      __syncthreads();  // (A) stage[cur] is complete; every warp has re-zeroed its rows; the previous frame's H stores are done
      if (tid == 0) {
        if (next_sig < gb) {  // this CTA's rows of the earlier blocks are written: announce them (release)
          __threadfence();
          for (int b = next_sig; b < gb; ++b) red_release_gpu_add(S.flags + ((size_t)cl * S.n_seq + b) * 2, 1);
        }
        if (gb >= S.TB && waited != gb) wait_flag_ge(S.flags + ((size_t)cl * S.n_seq + gb - S.TB) * 2 + 1, S.strips, S.stats ? S.stats + 1 : nullptr);
      }
      next_sig = gb;
      waited = gb;
      // S3: one thread per cell of the group's rows x Cc box, sums in table order
      const uint16_t* st = stage + cur * cap;
      for (int i = tid; i < ncell; i += NT_S) {
        const uint32_t cr = crec[i];
        const int eb = (int)((cr >> 11) & 0xFFFu), ee = eb + (int)(cr >> 23);
        float2 sr = make_float2(0.0f, 0.0f), si = make_float2(0.0f, 0.0f);
        for (int e = eb; e < ee; ++e) {
          float2 vr, vi;
          stage_to_pair(st[e], vr, vi);
          if constexpr (MODE == 0) {
            sr = __fadd2_rn(sr, vr); si = __fadd2_rn(si, vi);
          } else if constexpr (MODE == 1) {
            const float2 wv = tab2[e];
            sr = __ffma2_rn(vr, f2(wv.x), sr); sr = __ffma2_rn(neg2(vi), f2(wv.y), sr);
            si = __ffma2_rn(vi, f2(wv.x), si); si = __ffma2_rn(vr, f2(wv.y), si);
          } else {
            const float4 wv = tab4[e];
            const float2 wr = make_float2(wv.x, wv.y), wi = make_float2(wv.z, wv.w);
            sr = __ffma2_rn(vr, wr, sr); sr = __ffma2_rn(neg2(vi), wi, sr);
            si = __ffma2_rn(vi, wr, si); si = __ffma2_rn(vr, wi, si);
          }
        }
        buf[cr & 0x7FFu] = make_float4(sr.x, sr.y, si.x, si.y);
      }
      __syncthreads();  // (B) the rows are gridded; thread 0's wait above orders the H stores below after the consumers
      C2 z[16];
#pragma unroll
      for (int i = 0; i < 16; ++i) {  // step 1 inputs (prefold of the nbx elements that have a partner x + M)
        const int x = J * i + j;
        C2 a = to_c2(row[x]);
        if (x < P.nbx) {
          const C2 b = to_c2(row[x + M]);
          const float2 sg = f2(rho ? -1.0f : 1.0f);
          a.re = __ffma2_rn(b.re, sg, a.re); a.im = __ffma2_rn(b.im, sg, a.im);
        }
        z[bitrev4t(i)] = a;
      }
      __syncwarp();  // the row's 2 J threads (one warp) hold their inputs: its region becomes the exchange blocks
      {
        const float4* tw = tw1 + rho * TWV;
        const float4 t0 = tw[0];
        fft16_ramped(z, tw, t0.z, t0.w);
#pragma unroll
        for (int k1 = 0; k1 < 16; ++k1) xt[xsw(j, k1, rho)] = to_f4(z[k1]);
      }
      __syncwarp();
      float4* hrow = P.H + (((size_t)cl * S.Tring + slot) * t.R + y0 + r) * N + rho;
      if constexpr (J == 8) {
        C2 za[8], zb[8];
#pragma unroll
        for (int k = 0; k < 8; ++k) { za[bitrev3(k)] = to_c2(xt[xsw(k, j, rho)]); zb[bitrev3(k)] = to_c2(xt[xsw(k, j + 8, rho)]); }
        __syncwarp();  // exchange consumed: the row's region is zeroed for the next frame's gather
#pragma unroll
        for (int i = 0; i < N / (2 * J); ++i) row[lane % (2 * J) + i * 2 * J] = make_float4(0.0f, 0.0f, 0.0f, 0.0f);
        const float4 *ta = tw2 + (rho * 16 + j) * TWV, *tb = tw2 + (rho * 16 + j + 8) * TWV;
        const float4 a0 = ta[0], a1 = ta[1], b0 = tb[0], b1 = tb[1];
        fft8_ramped(za, a0.x, a0.y, a0.z, a0.w, a1.x, a1.y, a1.z, a1.w);
        fft8_ramped(zb, b0.x, b0.y, b0.z, b0.w, b1.x, b1.y, b1.z, b1.w);
        if (r < rows) {
#pragma unroll
          for (int k2 = 0; k2 < 8; ++k2) {
            __stcg(hrow + 2 * (j + 16 * k2), to_f4(za[k2]));
            __stcg(hrow + 2 * (j + 8 + 16 * k2), to_f4(zb[k2]));
          }
        }
      } else {
#pragma unroll
        for (int k = 0; k < 16; ++k) z[bitrev4t(k)] = to_c2(xt[xsw(k, j, rho)]);
        __syncwarp();
#pragma unroll
        for (int i = 0; i < N / (2 * J); ++i) row[lane % (2 * J) + i * 2 * J] = make_float4(0.0f, 0.0f, 0.0f, 0.0f);
        const float4* tw = tw2 + (rho * 16 + j) * TWV;
        const float4 t0 = tw[0];
        fft16_ramped(z, tw, t0.z, t0.w);
        if (r < rows) {
#pragma unroll
          for (int k2 = 0; k2 < 16; ++k2) __stcg(hrow + 2 * (j + 16 * k2), to_f4(z[k2]));
        }
      }
      if (p + S.K < S.n_pairs) put(cur ^ 1);
      cur ^= 1;
      pr += S.K;
      while (pr >= S.B) { pr -= S.B; ++pb; if (++rb == S.TB) rb = 0; }
    }
    __syncthreads();
    if (tid == 0) {  // every block of the wave is announced, also those in which this CTA had no frame
      __threadfence();
      for (int b = next_sig; b < (w + 1) * S.nbw; ++b) red_release_gpu_add(S.flags + ((size_t)cl * S.n_seq + b) * 2, 1);
    }
    next_sig = (w + 1) * S.nbw;
  }
}

// ---- consumer role: S4 along y + S5 + S6 for (channel slot cl, strip of W image columns), every wave,
// with the accumulators alive for the channel's whole time range; one CTA barrier per frame
template <int J, int NPROD>
__device__ __forceinline__ void stream_cols_role(const StreamParams& S, float4* tw1, float4* tw2, unsigned char* smem,
                                                 int cl, int strip) {
  constexpr int N = 32 * J, M = 16 * J, W = 64 / J, WP = W + 1;  // tile rows padded: a team's J rows fall in distinct bank groups
  const TiledParams& P = S.b;
  const DevTables& t = P.t;
  const int R = t.R, tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  float4* xbuf = reinterpret_cast<float4*>(smem);  // [2W teams][J * 16]
  float4* tile = xbuf + 2 * W * J * 16;            // [2][R + 1][WP]; row R stays zero
  const int tile_sz = (R + 1) * WP;
  const int rho = lane & 1, j = (lane >> 1) & (J - 1), w = warp * (16 / J) + lane / (2 * J);
  const int l0 = strip * W;
  float4* xt = xbuf + (2 * w + rho) * (J * 16);
  if (tid < 2 * WP) tile[(tid / WP) * tile_sz + R * WP + (tid % WP)] = make_float4(0.0f, 0.0f, 0.0f, 0.0f);
  const int* ready = S.flags + (size_t)cl * S.n_seq * 2;

  auto stage = [&](int slot, int b) {  // ring slot -> tile[b], 16 bytes per copy, L2 only
    const float4* src = P.H + (((size_t)cl * S.Tring + slot) * R) * N + l0;
    float4* dst = tile + b * tile_sz;
    for (int i = tid; i < R * W; i += NT_S) {
      const int y = i / W, ww = i - y * W;
      cp_async16(dst + y * WP + ww, src + (size_t)y * N + ww);
    }
    cp_async_commit();
  };

  for (int wv = 0; wv < S.n_waves; ++wv) {
    const int c = wv * S.Cw + cl;
    if (c >= P.n_chan) break;
    float2 acc[16], xy[NPROD == 4 ? 16 : 1];
#pragma unroll
    for (int k = 0; k < 16; ++k) acc[k] = make_float2(0.0f, 0.0f);
#pragma unroll
    for (int k = 0; k < (NPROD == 4 ? 16 : 1); ++k) xy[k] = make_float2(0.0f, 0.0f);
    const int gb0 = wv * S.nbw, n_prod = S.n_groups * S.K;
    if (tid == 0) wait_flag_ge(ready + (size_t)gb0 * 2, n_prod, S.stats);
    __syncthreads();  // the wave's first block is in the ring; the previous wave is done with the tiles
    int pb = 0, pr = 0, rb = gb0 % S.TB;  // block of the wave, frame in the block, ring block of frame p
    stage(rb * S.B, 0);
    for (int p = 0; p < S.n_pairs; ++p) {
      const int gb = gb0 + pb;
      const float4* cur = tile + (p & 1) * tile_sz;
      cp_async_wait_all();
      const bool next_new = p + 1 < S.n_pairs && pr + 1 == S.B;   // the prefetch below enters the next block
      if (tid == 0 && next_new) wait_flag_ge(ready + (size_t)(gb + 1) * 2, n_prod, S.stats);
      __syncthreads();  // this frame's tile is complete in shared memory; everybody is done with the other tile
      if (tid == 0 && (next_new || p + 1 == S.n_pairs)) {  // the block's last tile has been read: its ring slots may be reused
        __threadfence();
        red_release_gpu_add(S.flags + ((size_t)cl * S.n_seq + gb) * 2 + 1, 1);
      }
      if (++pr == S.B) { pr = 0; ++pb; if (++rb == S.TB) rb = 0; }  // now the position of frame p + 1
      if (p + 1 < S.n_pairs) stage(rb * S.B + pr, (p + 1) & 1);
      {  // step 1
        C2 z[16];
#pragma unroll
        for (int i = 0; i < 16; ++i) {
          const int y = J * i + j;
          const int ys = y < R ? y : R;  // rows beyond the occupied box: the zero row
          C2 a = to_c2(cur[ys * WP + w]);
          if (y < P.nby) {  // the few rows that have a partner y + M (prefold)
            const C2 b = to_c2(cur[(y + M) * WP + w]);
            const float2 sg = f2(rho ? -1.0f : 1.0f);
            a.re = __ffma2_rn(b.re, sg, a.re); a.im = __ffma2_rn(b.im, sg, a.im);
          }
          z[bitrev4t(i)] = a;
        }
        const float4* tw = tw1 + rho * TWV;
        const float4 t0 = tw[0];
        fft16_ramped(z, tw, t0.z, t0.w);
        __syncwarp();  // the team (same warp) has consumed the previous frame's exchange block
#pragma unroll
        for (int k1 = 0; k1 < 16; ++k1) xt[xsw(j, k1, rho)] = to_f4(z[k1]);
      }
      __syncwarp();
      if constexpr (J == 8) {  // step 2 + S5 + S6: k1 = j and j + 8
#pragma unroll
        for (int half = 0; half < 2; ++half) {
          C2 z[8];
          const int k1 = j + 8 * half;
#pragma unroll
          for (int k = 0; k < 8; ++k) z[bitrev3(k)] = to_c2(xt[xsw(k, k1, rho)]);
          const float4* tw = tw2 + (rho * 16 + k1) * TWV;
          const float4 a0 = tw[0], a1 = tw[1];
          fft8_ramped(z, a0.x, a0.y, a0.z, a0.w, a1.x, a1.y, a1.z, a1.w);
#pragma unroll
          for (int k2 = 0; k2 < 8; ++k2) accumulate_products<NPROD>(z[k2], acc[8 * half + k2], xy[NPROD == 4 ? 8 * half + k2 : 0]);
        }
      } else {
        C2 z[16];
#pragma unroll
        for (int k = 0; k < 16; ++k) z[bitrev4t(k)] = to_c2(xt[xsw(k, j, rho)]);
        const float4* tw = tw2 + (rho * 16 + j) * TWV;
        const float4 t0 = tw[0];
        fft16_ramped(z, tw, t0.z, t0.w);
#pragma unroll
        for (int k2 = 0; k2 < 16; ++k2) accumulate_products<NPROD>(z[k2], acc[k2], xy[NPROD == 4 ? k2 : 0]);
      }
    }
    // S6: one add per pixel per call; this CTA is the only writer of (channel c, columns l0 .. l0+W)
    const size_t plane = (size_t)N * N;
    float* o = P.out + (size_t)c * P.n_planes * plane + (l0 + w);
#pragma unroll
    for (int i = 0; i < 16; ++i) {
      const int k1 = (J == 8) ? j + 8 * (i >> 3) : j, k2 = (J == 8) ? (i & 7) : i;
      float* px = o + (size_t)(2 * (k1 + 16 * k2) + rho) * N;
      if constexpr (NPROD == 1) {
        px[0] += acc[i].x + acc[i].y;
      } else {
        px[0] += acc[i].x;
        px[plane] += acc[i].y;
      }
      if constexpr (NPROD == 4) {  // YX = conj(XY)
        px[2 * plane] += xy[i].x;
        px[3 * plane] += xy[i].y;
        px[4 * plane] += xy[i].x;
        px[5 * plane] -= xy[i].y;
      }
    }
  }
}

template <int J, int NPROD, int MODE>
__global__ void __launch_bounds__(NT_S, 3) tiled_stream(StreamParams S) {
  extern __shared__ __align__(16) unsigned char smem_raw[];
  float4* tw1 = reinterpret_cast<float4*>(smem_raw);  // [2][TWV]
  float4* tw2 = tw1 + 2 * TWV;                        // [2][16][TWV]
  unsigned char* rest = reinterpret_cast<unsigned char*>(tw2 + 2 * 16 * TWV);
  for (int i = threadIdx.x; i < 2 * TWV; i += NT_S) tw1[i] = __ldg(S.b.tw1 + i);
  for (int i = threadIdx.x; i < 2 * 16 * TWV; i += NT_S) tw2[i] = __ldg(S.b.tw2 + i);
  const int n_cols = S.Cw * S.strips;
  const long long t_begin = clock64();
  if ((int)blockIdx.x < n_cols) {
    stream_cols_role<J, NPROD>(S, tw1, tw2, rest, (int)blockIdx.x / S.strips, (int)blockIdx.x % S.strips);
    if (S.stats && threadIdx.x == 0) atomicAdd(S.stats + 2, (unsigned long long)(clock64() - t_begin));
  } else {
    const int rr = (int)blockIdx.x - n_cols, per_chan = S.n_groups * S.K;
    const int cl = rr / per_chan, gk = rr - cl * per_chan;
    stream_rows_role<J, MODE>(S, tw1, tw2, rest, cl, gk / S.K, gk % S.K);
    if (S.stats && threadIdx.x == 0) atomicAdd(S.stats + 3, (unsigned long long)(clock64() - t_begin));
  }
}

struct TiledTables {
  float4* tw1;
  float4* tw2;
  float4* ent_rec;
};

template <int J>
size_t rows_smem_bytes(int n_ant) {
  constexpr int N = 32 * J, RG = NT_A<J> / (2 * J), XS = x_team_stride<J>();
  constexpr int BUF = (RG * N > 2 * RG * XS) ? RG * N : 2 * RG * XS;
  return ((size_t)BUF + 2 * TWV + 2 * 16 * TWV) * sizeof(float4) + (size_t)n_ant * sizeof(uint32_t);
}
template <int J>
size_t cols_smem_bytes(int R) {
  constexpr int W = 64 / J, XS = x_team_stride_cols<J>();
  return ((size_t)2 * W * XS + 2 * TWV + 2 * 16 * TWV + (size_t)2 * (R + 1) * W) * sizeof(float4);
}

template <typename K>
int set_dyn_smem(K kern, size_t bytes) {
  if (bytes > 48 * 1024)
    EPIC_CUDA_TRY(cudaFuncSetAttribute((const void*)kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)bytes));
  return EPIC_OK;
}

template <int J, int NPROD>
int launch_cols(const TiledParams& P, dim3 grid, size_t smem, cudaStream_t s) {
  int st = set_dyn_smem(tiled_cols<J, NPROD>, smem);
  if (st != EPIC_OK) return st;
  tiled_cols<J, NPROD><<<grid, NT_B, smem, s>>>(P);
  return EPIC_OK;
}

template <int J, int NPROD>
int cols_occupancy(int* occ, size_t smem) {
  int st = set_dyn_smem(tiled_cols<J, NPROD>, smem);
  if (st != EPIC_OK) return st;
  EPIC_CUDA_TRY(cudaOccupancyMaxActiveBlocksPerMultiprocessor(occ, tiled_cols<J, NPROD>, NT_B, smem));
  return EPIC_OK;
}

template <int J>
int tiled_image_j(epic_plan* p, const ImageArgs& a, TiledParams& P) {
  constexpr int N = 32 * J, W = 64 / J, RG = NT_A<J> / (2 * J);
  const int R = p->R;
  const int n_pairs = a.n_pol == 2 ? a.n_t : (a.n_t + 1) / 2;
  const size_t frame_bytes = (size_t)R * N * sizeof(float4);
  const long long max_frames = (long long)std::max<size_t>(1, scratch_budget(p) / frame_bytes);
  const int strips = N / W;
  const size_t smem_a = rows_smem_bytes<J>(p->n_ant), smem_b = cols_smem_bytes<J>(R);
  const bool delta = p->t.is_delta != 0;
  int st = delta ? set_dyn_smem(tiled_rows<J, true>, smem_a) : set_dyn_smem(tiled_rows<J, false>, smem_a);
  if (st != EPIC_OK) return st;
  // both kernels run as ONE wave: strips x Cb column CTAs, and an equal share of the row items per CTA
  int occ_a = 0, occ_b = 0;
  if (delta) EPIC_CUDA_TRY(cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ_a, tiled_rows<J, true>, NT_A<J>, smem_a));
  else EPIC_CUDA_TRY(cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ_a, tiled_rows<J, false>, NT_A<J>, smem_a));
  if (a.n_products == 1) st = cols_occupancy<J, 1>(&occ_b, smem_b);
  else if (a.n_products == 2) st = cols_occupancy<J, 2>(&occ_b, smem_b);
  else st = cols_occupancy<J, 4>(&occ_b, smem_b);
  if (st != EPIC_OK) return st;
  if (occ_a < 1 || occ_b < 1) return EPIC_ERR_RANGE;
  long long Cb = std::min<long long>(a.n_chan, ((long long)occ_b * p->n_sm) / strips);
  Cb = std::max<long long>(1, std::min(Cb, max_frames));
  const long long Tb = std::max<long long>(1, std::min<long long>(n_pairs, max_frames / Cb));
  const int n_groups = (R + RG - 1) / RG;
  int launches = 0;
  for (int c0 = 0; c0 < a.n_chan; c0 += (int)Cb) {
    P.c0 = c0;
    P.Cb = (int)std::min<long long>(Cb, a.n_chan - c0);
    for (int p0 = 0; p0 < n_pairs; p0 += (int)Tb) {
      P.p0 = p0;
      P.Tb = (int)std::min<long long>(Tb, n_pairs - p0);
      const long long items = (long long)P.Cb * P.Tb * n_groups;
      const dim3 grid_a((unsigned)std::min<long long>(items, (long long)occ_a * p->n_sm));
      if (delta) tiled_rows<J, true><<<grid_a, NT_A<J>, smem_a, a.stream>>>(P);
      else tiled_rows<J, false><<<grid_a, NT_A<J>, smem_a, a.stream>>>(P);
      const dim3 grid_b(strips, P.Cb);
      if (a.n_products == 1) st = launch_cols<J, 1>(P, grid_b, smem_b, a.stream);
      else if (a.n_products == 2) st = launch_cols<J, 2>(P, grid_b, smem_b, a.stream);
      else st = launch_cols<J, 4>(P, grid_b, smem_b, a.stream);
      if (st != EPIC_OK) return st;
      launches += 2;
    }
  }
  EPIC_CUDA_TRY(cudaGetLastError());
  p->last_launches = launches;
  return EPIC_OK;
}

// ---- host side of the streamed variant
constexpr size_t STREAM_RING_DEFAULT = (size_t)40 << 20;  // ring of row-transformed frames: well inside the 126 MB L2

template <int J>
size_t stream_rows_bytes(int mode, int cap, int Cc) {
  const size_t ent = mode == 0 ? stream_ent_bytes<0>() : (mode == 1 ? stream_ent_bytes<1>() : stream_ent_bytes<2>());
  return (size_t)stream_rg<J>() * 32 * J * sizeof(float4) + (size_t)cap * ent + (size_t)stream_rg<J>() * Cc * sizeof(uint32_t);
}
template <int J>
size_t stream_cols_bytes(int R) {
  constexpr int W = 64 / J;
  return ((size_t)2 * W * J * 16 + (size_t)2 * (R + 1) * (W + 1)) * sizeof(float4);
}
template <int J>
size_t stream_smem_bytes(int mode, int cap, int R, int Cc) {
  const size_t tw = (size_t)(2 * TWV + 2 * 16 * TWV) * sizeof(float4);
  return tw + ((std::max(stream_rows_bytes<J>(mode, cap, Cc), stream_cols_bytes<J>(R)) + 15) & ~(size_t)15);
}

// most gather entries in one group of RG occupied rows, over all layouts
int stream_max_group_entries(const epic_plan* p, int RG) {
  size_t best = 0;
  for (int l = 0; l < p->n_layout; ++l) {
    std::vector<size_t> per((size_t)(p->R + RG - 1) / RG, 0);
    for (uint32_t i = p->h_cell_off[l]; i < p->h_cell_off[l + 1]; ++i) {
      per[p->h_cells[i].y / RG] += p->h_cells[i].ent_count;
      if (p->h_cells[i].ent_count > 511u) return 1 << 30;  // a row CTA's cell record holds 9 bits of entry count
    }
    for (size_t v : per) best = std::max(best, v);
  }
  return (int)std::min<size_t>(best, (size_t)1 << 30);
}

template <int J, int NPROD, int MODE>
int launch_stream(epic_plan* p, const ImageArgs& a, StreamParams& S, int cap) {
  const int R = p->R, n_groups = (R + stream_rg<J>() - 1) / stream_rg<J>(), strips = (32 * J) / (64 / J);
  const size_t smem = stream_smem_bytes<J>(MODE, cap, R, p->Cc);
  auto kern = tiled_stream<J, NPROD, MODE>;
  if (smem > (size_t)226 * 1024) return EPIC_ERR_RANGE;
  EPIC_CUDA_TRY(cudaFuncSetAttribute((const void*)kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
  int per_sm = 0;
  EPIC_CUDA_TRY(cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, kern, NT_S, smem));
  const long long slots = (long long)per_sm * p->n_sm;
  // K row CTAs per (channel, row group), interleaved in time: a row item is a longer dependent chain than a column
  // frame, and rows : columns = K n_groups : strips is then close to the 1 : 1 split of the work
  int K = 2;  // measured on C4 / C5: K = 1 1.40 / 0.094, K = 2 1.95 / 0.216, K = 3 1.65 / (falls back to 1) M frames/s
  if (slots / (strips + K * n_groups) < 1) K = 1;
  long long Cw = std::min<long long>(a.n_chan, slots / (strips + K * n_groups));
  if (Cw < 1) return EPIC_ERR_RANGE;
  const int n_waves = (int)((a.n_chan + Cw - 1) / Cw);
  Cw = (a.n_chan + n_waves - 1) / n_waves;  // equal waves
  const int n_pairs = a.n_pol == 2 ? a.n_t : (a.n_t + 1) / 2;
  int B = 4;  // frames per hand-over block: one flag round trip per B frames (measured: 1, 4, 8 within 6 % of each other)
  B = std::min(B, n_pairs);
  const int nbw = (n_pairs + B - 1) / B;
  const long long n_seq = (long long)n_waves * nbw;
  const size_t flag_bytes = (((size_t)Cw * n_seq * 2 * sizeof(int)) + 255) & ~(size_t)255;
  const size_t frame_bytes = (size_t)R * 32 * J * sizeof(float4);
  // the ring: scratch_limit (if set) or the default, at least two blocks per channel, inside the plan's scratch
  const size_t budget = p->scratch_bytes;
  if (flag_bytes + (size_t)2 * B * Cw * frame_bytes > budget) return EPIC_ERR_RANGE;
  const size_t ring = std::min(budget - flag_bytes, p->scratch_limit ? p->scratch_limit : STREAM_RING_DEFAULT);
  long long TB = (long long)(ring / ((size_t)Cw * frame_bytes * B));  // ring length in blocks, >= 2 (see the roles' waits)
  TB = std::max<long long>(2, std::min<long long>(TB, 16));
  const long long Tring = TB * B;
  S.flags = static_cast<int*>(p->d_scratch);
  S.b.H = reinterpret_cast<float4*>(static_cast<char*>(p->d_scratch) + flag_bytes);
  S.Cw = (int)Cw;
  S.n_waves = n_waves;
  S.n_pairs = n_pairs;
  S.n_seq = (int)n_seq;
  S.Tring = (int)Tring;
  S.B = B;
  S.nbw = nbw;
  S.TB = (int)TB;
  S.n_groups = n_groups;
  S.strips = strips;
  S.ent_cap = cap;
  S.K = K;
  EPIC_CUDA_TRY(cudaMemsetAsync(S.flags, 0, flag_bytes, a.stream));
  const bool want_stats = std::getenv("EPIC_STREAM_STATS") != nullptr;  // development: role wait / total cycles on stderr
  S.stats = nullptr;
  if (want_stats) {
    EPIC_CUDA_TRY(cudaMalloc(&S.stats, 4 * sizeof(unsigned long long)));
    EPIC_CUDA_TRY(cudaMemsetAsync(S.stats, 0, 4 * sizeof(unsigned long long), a.stream));
  }
  void* args[] = {&S};
  const dim3 grid((unsigned)(Cw * (strips + K * n_groups)));
  EPIC_CUDA_TRY(cudaLaunchCooperativeKernel((const void*)kern, grid, dim3(NT_S), args, smem, a.stream));
  if (want_stats) {
    unsigned long long h[4];
    EPIC_CUDA_TRY(cudaMemcpy(h, S.stats, sizeof(h), cudaMemcpyDeviceToHost));
    cudaFree(S.stats);
    const double nc = (double)Cw * strips, nr = (double)Cw * K * n_groups;
    fprintf(stderr, "stream stats: Cw %lld K %d B %d TB %lld waves %d | cols wait %.0f of %.0f kcyc per CTA | rows wait %.0f of %.0f kcyc per CTA\n",
            Cw, K, B, TB, n_waves, h[0] / nc / 1e3, h[2] / nc / 1e3, h[1] / nr / 1e3, h[3] / nr / 1e3);
  }
  p->last_launches = 1;
  return EPIC_OK;
}

template <int J>
int stream_image_j(epic_plan* p, const ImageArgs& a, StreamParams& S) {
  const int cap = (std::max(stream_max_group_entries(p, stream_rg<J>()), 8) + 7) & ~7;
  if (cap > PF_MAX * NT_S) return EPIC_ERR_RANGE;
  const int mode = a.phasor_pair ? 2 : (p->t.is_delta ? 0 : 1);
#define EPIC_STREAM_CASE(NPROD)                                                   \
  (mode == 0 ? launch_stream<J, NPROD, 0>(p, a, S, cap)                           \
             : (mode == 1 ? launch_stream<J, NPROD, 1>(p, a, S, cap) : launch_stream<J, NPROD, 2>(p, a, S, cap)))
  if (a.n_products == 1) return EPIC_STREAM_CASE(1);
  if (a.n_products == 2) return EPIC_STREAM_CASE(2);
  return EPIC_STREAM_CASE(4);
#undef EPIC_STREAM_CASE
}

}  // namespace

int stream_supported(const epic_plan* p, int is_cf32, int n_pol, int n_products) {
  if (!p->tiled_ok || is_cf32) return 0;
  if (!((n_pol == 1 && n_products == 1) || (n_pol == 2 && (n_products == 2 || n_products == 4)))) return 0;
  const int J = p->N / 32, RG = NT_S / (2 * J);
  const int cap = (std::max(stream_max_group_entries(p, RG), 8) + 7) & ~7;
  if (cap > PF_MAX * NT_S) return 0;
  const int mode = p->d_phasor_pair ? 2 : (p->t.is_delta ? 0 : 1);
  const size_t smem = J == 8 ? stream_smem_bytes<8>(mode, cap, p->R, p->Cc) : stream_smem_bytes<16>(mode, cap, p->R, p->Cc);
  if (smem > (size_t)226 * 1024) return 0;
  // at least one channel's column strips and row groups must be co-resident
  const long long per_sm = std::min<long long>(3, ((size_t)227 * 1024) / (smem + 1024));
  const int strips = p->N / (64 / J), n_groups = (p->R + RG - 1) / RG;
  return per_sm * p->n_sm >= strips + n_groups ? 1 : 0;
}

int stream_image(epic_plan* p, const ImageArgs& a) {
  const TiledTables* tt = static_cast<const TiledTables*>(p->d_tiled);
  StreamParams S;
  TiledParams& P = S.b;
  P.t = p->t;
  P.volt = static_cast<const uint8_t*>(a.volt);
  P.H = nullptr;
  P.out = a.out;
  P.tw1 = tt->tw1;
  P.tw2 = tt->tw2;
  P.ent_rec = tt->ent_rec;
  P.native = a.native;
  P.phasor = a.phasor_pair;
  P.n_t = a.n_t;
  P.n_chan = a.n_chan;
  P.n_pol = a.n_pol;
  P.n_planes = a.n_planes;
  P.c0 = P.p0 = P.Cb = P.Tb = 0;
  P.nbx = std::max(0, p->Cc - p->N / 2);
  P.nby = std::max(0, p->R - p->N / 2);
  return p->N == 256 ? stream_image_j<8>(p, a, S) : stream_image_j<16>(p, a, S);
}

// ---------------------------------------------------------------- host side
int tiled_plan_init(epic_plan* p) {
  p->tiled_ok = 0;
  p->d_tiled = nullptr;
  if (p->N != 256 && p->N != 512) return EPIC_OK;
  const int N = p->N, J = N / 32, M = N / 2;
  // twiddles from double (reading Q8: + sign).  ramped16(q): the TwSet words of base q = exp(i ang)
  auto cis = [](double ang, float* re, float* im) { *re = (float)std::cos(ang); *im = (float)std::sin(ang); };
  auto ramped16 = [&](double ang, float4* out) {
    float v[20] = {0};
    v[0] = 1.0f;                                                                       // fold constant unused here
    cis(8.0 * ang, &v[2], &v[3]);                                                      // level 2: q^8
    cis(4.0 * ang, &v[4], &v[5]);                                                      // level 4: q^4
    for (int k = 0; k < 2; ++k) cis(2.0 * ang + 2.0 * M_PI * k / 8.0, &v[6 + 2 * k], &v[7 + 2 * k]);     // q^2 W_8^k
    for (int k = 0; k < 4; ++k) cis(ang + 2.0 * M_PI * k / 16.0, &v[10 + 2 * k], &v[11 + 2 * k]);        // q W_16^k
    for (int w = 0; w < TWV; ++w) out[w] = make_float4(v[4 * w], v[4 * w + 1], v[4 * w + 2], v[4 * w + 3]);
  };
  auto ramped8 = [&](double ang, float4* out) {
    float v[20] = {0};
    cis(4.0 * ang, &v[0], &v[1]);                                                      // level 2: q^4
    cis(2.0 * ang, &v[2], &v[3]);                                                      // level 4: q^2
    for (int k = 0; k < 2; ++k) cis(ang + 2.0 * M_PI * k / 8.0, &v[4 + 2 * k], &v[5 + 2 * k]);           // q W_8^k
    for (int w = 0; w < TWV; ++w) out[w] = make_float4(v[4 * w], v[4 * w + 1], v[4 * w + 2], v[4 * w + 3]);
  };
  std::vector<float4> tw1((size_t)2 * TWV), tw2((size_t)2 * 16 * TWV);
  for (int rho = 0; rho < 2; ++rho) {
    const double r_ang = 2.0 * M_PI * (double)rho / (double)N;
    ramped16(r_ang * J, &tw1[(size_t)rho * TWV]);                                     // step 1: base r^J
    for (int k1 = 0; k1 < 16; ++k1) {
      const double q_ang = r_ang + 2.0 * M_PI * (double)k1 / (double)M;               // step 2: base r W_M^{k1}
      if (J == 16) ramped16(q_ang, &tw2[((size_t)rho * 16 + k1) * TWV]);
      else ramped8(q_ang, &tw2[((size_t)rho * 16 + k1) * TWV]);
    }
  }
  TiledTables* tt = new (std::nothrow) TiledTables();
  if (!tt) return EPIC_ERR_NOMEM;
  std::vector<float4> rec(std::max<size_t>(1, p->h_ent_ant.size()));
  for (size_t e = 0; e < p->h_ent_ant.size(); ++e) {
    const uint32_t ant = p->h_ent_ant[e];
    float antf;
    std::memcpy(&antf, &ant, sizeof(float));
    rec[e] = make_float4(p->h_ent_tap[e].x, p->h_ent_tap[e].y, antf, 0.0f);
  }
  tt->tw1 = tt->tw2 = tt->ent_rec = nullptr;
  cudaError_t ce = cudaMalloc(&tt->tw1, tw1.size() * sizeof(float4));
  if (ce == cudaSuccess) ce = cudaMalloc(&tt->ent_rec, rec.size() * sizeof(float4));
  if (ce == cudaSuccess) ce = cudaMemcpy(tt->ent_rec, rec.data(), rec.size() * sizeof(float4), cudaMemcpyHostToDevice);
  if (ce == cudaSuccess) ce = cudaMalloc(&tt->tw2, tw2.size() * sizeof(float4));
  if (ce == cudaSuccess) ce = cudaMemcpy(tt->tw1, tw1.data(), tw1.size() * sizeof(float4), cudaMemcpyHostToDevice);
  if (ce == cudaSuccess) ce = cudaMemcpy(tt->tw2, tw2.data(), tw2.size() * sizeof(float4), cudaMemcpyHostToDevice);
  if (ce != cudaSuccess) {
    set_cuda_error(ce);
    if (tt->tw1) cudaFree(tt->tw1);
    if (tt->tw2) cudaFree(tt->tw2);
    if (tt->ent_rec) cudaFree(tt->ent_rec);
    delete tt;
    return ce == cudaErrorMemoryAllocation ? EPIC_ERR_NOMEM : EPIC_ERR_CUDA;
  }
  p->d_tiled = tt;
  p->tiled_ok = 1;
  return EPIC_OK;
}

void tiled_plan_free(epic_plan* p) {
  TiledTables* tt = static_cast<TiledTables*>(p->d_tiled);
  if (tt) {
    if (tt->tw1) cudaFree(tt->tw1);
    if (tt->tw2) cudaFree(tt->tw2);
    if (tt->ent_rec) cudaFree(tt->ent_rec);
    delete tt;
  }
  p->d_tiled = nullptr;
  p->tiled_ok = 0;
}

int tiled_supported(const epic_plan* p, int is_cf32, int n_pol, int n_products) {
  if (!p->tiled_ok || is_cf32) return 0;
  if (!((n_pol == 1 && n_products == 1) || (n_pol == 2 && (n_products == 2 || n_products == 4)))) return 0;
  if (p->n_ant % 4 != 0) return 0;  // voltage rows are read as 32-bit words
  const size_t smem_a = p->N == 256 ? rows_smem_bytes<8>(p->n_ant) : rows_smem_bytes<16>(p->n_ant);
  const size_t smem_b = p->N == 256 ? cols_smem_bytes<8>(p->R) : cols_smem_bytes<16>(p->R);
  return (smem_a <= (size_t)220 * 1024 && smem_b <= (size_t)220 * 1024) ? 1 : 0;
}

int tiled_image(epic_plan* p, const ImageArgs& a) {
  const TiledTables* tt = static_cast<const TiledTables*>(p->d_tiled);
  TiledParams P;
  P.t = p->t;
  P.volt = static_cast<const uint8_t*>(a.volt);
  P.H = static_cast<float4*>(p->d_scratch);
  P.out = a.out;
  P.tw1 = tt->tw1;
  P.tw2 = tt->tw2;
  P.ent_rec = tt->ent_rec;
  P.native = a.native;
  P.phasor = a.phasor_pair;
  P.n_t = a.n_t;
  P.n_chan = a.n_chan;
  P.n_pol = a.n_pol;
  P.n_planes = a.n_planes;
  P.nbx = std::max(0, p->Cc - p->N / 2);
  P.nby = std::max(0, p->R - p->N / 2);
  return p->N == 256 ? tiled_image_j<8>(p, a, P) : tiled_image_j<16>(p, a, P);
}

}  // namespace epic
