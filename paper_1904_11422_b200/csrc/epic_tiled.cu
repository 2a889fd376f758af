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

}  // namespace

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
