// Fused EPIC path: unpack -> grid -> 2-D transform -> products -> accumulate in ONE kernel, the
// aperture/image planes never leave the SM (BASELINE.json north_star (1)-(4)).
//
// Applies when the occupied cells of the aperture fit a 32 x 32 box (after the circular
// relocation of epic_plan.cu; SURVEY.md reading Q7) and N = 32*Q, Q in {1,2,4,8}.  With the
// support S = 32 cells a side, the N x N image splits into Q*Q independent 32 x 32 sub-images
//
//   A[Q m1 + m2][Q l1 + l2] = sum_{y,x<32} G[y][x] W_N^{x l2} W_N^{y m2} W_32^{x l1 + y m1},
//
// i.e. the zero rows/columns of the padded plane are never transformed (a pruned decimation-in-
// frequency 2-D FFT: the first log2 Q stages of each axis only multiply by a phase ramp).
// Work unit = (channel c, column residue l2); its CTA owns the image columns l = Q l1 + l2 and
// keeps their accumulators in registers for the whole integration:
//
//   per batch of Q frames:
//     stage    cp.async the next batch's 4+4-bit voltages into shared memory (double buffer)
//     gather   S1+S3: every thread owns fixed cells of the 32x32 block and sums its (antenna, tap)
//              list in table order (no atomics, deterministic) for all frames/pols of the batch
//     rows     S4 along x: one thread per (frame, pol, row): 32 inputs -> the 32 outputs l1 of
//              this CTA's l2, in registers, written back in place
//     columns  S4 along y + S5 + S6: one thread per (pol, m2, l1): 32 inputs from shared memory ->
//              32 outputs m1 in registers -> products -> += register accumulators
//   at the end of the unit's frames: one atomicAdd per pixel into out_accum.
//
// The 32-point transforms run as TWO 16-point FFTs packed in the halves of f32x2 registers
// (sm_100 FFMA2/FADD2): outputs 2Q k + rho for rho = m2 (low half) and m2 + Q (high half),
// k = 0..15, of   X[2Q k + rho] = sum_{y<16} (in[y] W_N^{y rho} + in[y+16] W_N^{(y+16) rho}) W_16^{y k}.
// The bracket ("fold + ramp") is scalar FP32 with compile-time twiddles; the 16-point FFT is
// radix-2 decimation-in-time with the 6-FMA butterfly, twiddles as immediates.
#include <algorithm>

#include "epic_internal.h"

namespace epic {
namespace {

constexpr int S = 32;   // support block side (cells)
constexpr int HS = 34;  // row stride of the shared planes, complex elements (16-byte rows, conflict-free)

// ---------------------------------------------------------------- compile-time twiddles
// exp(+2 pi i ex / n) in double, evaluated by the compiler (reading Q8: + sign, inverse DFT).
constexpr double kPi = 3.14159265358979323846264338327950288;
constexpr double sin_small(double x) {
  const double x2 = x * x;
  double term = x, sum = x;
  for (int i = 1; i <= 12; ++i) { term *= -x2 / (double)((2 * i) * (2 * i + 1)); sum += term; }
  return sum;
}
constexpr double cos_small(double x) {
  const double x2 = x * x;
  double term = 1.0, sum = 1.0;
  for (int i = 1; i <= 12; ++i) { term *= -x2 / (double)((2 * i - 1) * (2 * i)); sum += term; }
  return sum;
}
constexpr int mod_pos(int a, int n) { return ((a % n) + n) % n; }
constexpr double tw_cos(int ex, int n) {
  ex = mod_pos(ex, n);
  const int j = (4 * ex + n / 2) / n;  // nearest quarter turn
  const double phi = 2.0 * kPi * (double)(4 * ex - j * n) / (4.0 * (double)n);
  const double cs = cos_small(phi), sn = sin_small(phi);
  switch (j & 3) { case 0: return cs; case 1: return -sn; case 2: return -cs; default: return sn; }
}
constexpr double tw_sin(int ex, int n) {
  ex = mod_pos(ex, n);
  const int j = (4 * ex + n / 2) / n;
  const double phi = 2.0 * kPi * (double)(4 * ex - j * n) / (4.0 * (double)n);
  const double cs = cos_small(phi), sn = sin_small(phi);
  switch (j & 3) { case 0: return sn; case 1: return cs; case 2: return -sn; default: return -cs; }
}
constexpr int bitrev4(int v) { return ((v & 1) << 3) | ((v & 2) << 1) | ((v & 4) >> 1) | ((v & 8) >> 3); }

// ---------------------------------------------------------------- packed complex pair
// (lo, hi) halves hold two independent 16-point transforms (rho = r and r + Q).
struct C2 { float2 re, im; };

__device__ __forceinline__ float2 f2(float v) { return make_float2(v, v); }
__device__ __forceinline__ float2 neg2(float2 v) { return make_float2(-v.x, -v.y); }

// acc += v * exp(2 pi i EX / NN), scalar, compile-time twiddle
template <int EX, int NN>
__device__ __forceinline__ void cmadd(float& ar, float& ai, float vr, float vi) {
  constexpr int e = mod_pos(EX, NN);
  if constexpr (e == 0) { ar += vr; ai += vi; }
  else if constexpr (4 * e == NN) { ar -= vi; ai += vr; }
  else if constexpr (2 * e == NN) { ar -= vr; ai -= vi; }
  else if constexpr (4 * e == 3 * NN) { ar += vi; ai -= vr; }
  else {
    constexpr float wr = (float)tw_cos(e, NN), wi = (float)tw_sin(e, NN);
    ar = fmaf(vr, wr, ar); ar = fmaf(-vi, wi, ar);
    ai = fmaf(vi, wr, ai); ai = fmaf(vr, wi, ai);
  }
}
// v * exp(2 pi i EX / NN)
template <int EX, int NN>
__device__ __forceinline__ void cmul_tw(float& outr, float& outi, float vr, float vi) {
  constexpr int e = mod_pos(EX, NN);
  if constexpr (e == 0) { outr = vr; outi = vi; }
  else if constexpr (4 * e == NN) { outr = -vi; outi = vr; }
  else if constexpr (2 * e == NN) { outr = -vr; outi = -vi; }
  else if constexpr (4 * e == 3 * NN) { outr = vi; outi = -vr; }
  else {
    constexpr float wr = (float)tw_cos(e, NN), wi = (float)tw_sin(e, NN);
    outr = fmaf(-vi, wi, vr * wr);
    outi = fmaf(vr, wi, vi * wr);
  }
}

// radix-2 DIT butterfly on packed pairs: (a, b) <- (a + w b, a - w b), w = exp(2 pi i K / NN)
template <int K, int NN>
__device__ __forceinline__ void bfly(C2& a, C2& b) {
  if constexpr (K == 0) {
    const C2 p = {__fadd2_rn(a.re, b.re), __fadd2_rn(a.im, b.im)};
    b.re = __fadd2_rn(a.re, neg2(b.re)); b.im = __fadd2_rn(a.im, neg2(b.im));
    a = p;
  } else if constexpr (4 * K == NN) {  // w = +i: w b = (-b.im, b.re)
    const C2 p = {__fadd2_rn(a.re, neg2(b.im)), __fadd2_rn(a.im, b.re)};
    const C2 q = {__fadd2_rn(a.re, b.im), __fadd2_rn(a.im, neg2(b.re))};
    a = p; b = q;
  } else {
    constexpr float wr = (float)tw_cos(K, NN), wi = (float)tw_sin(K, NN);
    C2 p;
    p.re = __ffma2_rn(b.re, f2(wr), a.re); p.re = __ffma2_rn(neg2(b.im), f2(wi), p.re);
    p.im = __ffma2_rn(b.im, f2(wr), a.im); p.im = __ffma2_rn(b.re, f2(wi), p.im);
    b.re = __ffma2_rn(a.re, f2(2.0f), neg2(p.re));
    b.im = __ffma2_rn(a.im, f2(2.0f), neg2(p.im));
    a = p;
  }
}

template <int NN, int BASE, int K>
__device__ __forceinline__ void fft16_block(C2 (&z)[16]) {
  if constexpr (K < NN / 2) {
    bfly<K, NN>(z[BASE + K], z[BASE + K + NN / 2]);
    fft16_block<NN, BASE, K + 1>(z);
  }
}
template <int NN, int BASE>
__device__ __forceinline__ void fft16_stage(C2 (&z)[16]) {
  if constexpr (BASE < 16) {
    fft16_block<NN, BASE, 0>(z);
    fft16_stage<NN, BASE + NN>(z);
  }
}
// z holds the input in bit-reversed order; on return z[k] = sum_y in[y] exp(+2 pi i y k / 16).
__device__ __forceinline__ void fft16(C2 (&z)[16]) {
  fft16_stage<2, 0>(z);
  fft16_stage<4, 0>(z);
  fft16_stage<8, 0>(z);
  fft16_stage<16, 0>(z);
}

// fold + ramp for input pair (y, y+16) of residue pair (RHO, RHO+Q), N = 32 Q
template <int Q, int RHO, int Y>
__device__ __forceinline__ void fold_one(C2 (&z)[16], float2 a, float2 b, bool has_b) {
  constexpr int N = 32 * Q;
  float lr, li, hr, hi;
  cmul_tw<Y * RHO, N>(lr, li, a.x, a.y);
  cmul_tw<Y * (RHO + Q), N>(hr, hi, a.x, a.y);
  if (has_b) {
    cmadd<(Y + 16) * RHO, N>(lr, li, b.x, b.y);
    cmadd<(Y + 16) * (RHO + Q), N>(hr, hi, b.x, b.y);
  }
  z[bitrev4(Y)].re = make_float2(lr, hr);
  z[bitrev4(Y)].im = make_float2(li, hi);
}
template <int Q, int RHO, int Y>
__device__ __forceinline__ void fold_all(C2 (&z)[16], const float2* __restrict__ in, int stride, int n_valid) {
  if constexpr (Y < 16) {
    const float2 zero = make_float2(0.0f, 0.0f);
    const float2 a = (Y < n_valid) ? in[Y * stride] : zero;
    const bool has_b = (Y + 16 < n_valid);
    const float2 b = has_b ? in[(Y + 16) * stride] : zero;
    fold_one<Q, RHO, Y>(z, a, b, has_b);
    fold_all<Q, RHO, Y + 1>(z, in, stride, n_valid);
  }
}

// The 32-point pruned transform of this file's header: in[y], y < n_valid (<= 32), zero beyond.
// z[k].lo = X[2Q k + RHO], z[k].hi = X[2Q k + RHO + Q].
template <int Q, int RHO>
__device__ __forceinline__ void dft32_pair(C2 (&z)[16], const float2* __restrict__ in, int stride, int n_valid) {
  fold_all<Q, RHO, 0>(z, in, stride, n_valid);
  fft16(z);
}

// ---------------------------------------------------------------- kernel parameters
struct FusedParams {
  const uint8_t* volt;       // [T][C][NPOL][A] 4+4-bit samples
  float* out;                // [C][planes][N][N]
  const uint32_t* cell_info; // [32*32] dense block cells: (first entry << 8) | entry count
  const uint16_t* ent_ant;   // gather entries, sorted by block cell
  const float2* ent_tap;
  int n_t, n_chan, n_ant, n_planes;
  int R, Cc;                 // occupied rows / columns of the block
  int nb;                    // batches per unit = ceil(n_t / Q)
  long long total;           // n_chan * Q * nb batches in all
  int row_bytes;             // NPOL * A
  int row_pitch;             // row_bytes rounded up to 16
  int aligned16;             // voltages can be staged with 16-byte cp.async
};

__device__ __forceinline__ void cp_async16(void* smem_dst, const void* gmem_src) {
  const unsigned d = (unsigned)__cvta_generic_to_shared(smem_dst);
  asm volatile("cp.async.cg.shared.global [%0], [%1], 16;" ::"r"(d), "l"(gmem_src) : "memory");
}
__device__ __forceinline__ void cp_async_commit() { asm volatile("cp.async.commit_group;" ::: "memory"); }
__device__ __forceinline__ void cp_async_wait_all() { asm volatile("cp.async.wait_group 0;" ::: "memory"); }

// S1 (reading Q1): byte hhhhllll -> ((h ^ 8) << 16) | (l ^ 8), i.e. both
// two's-complement nibbles biased by +8 in the halves of one word, so a cell's samples can be
// summed with one integer add.
__device__ __forceinline__ uint32_t unpack_biased(uint32_t byte) {
  return ((byte * 0x1001u) & 0x000F000Fu) ^ 0x00080008u;
}
__device__ __forceinline__ float small_int_to_float(int v) {  // exact for |v| < 2^22, no I2F
  return __int_as_float(0x4B400000 + v) - 12582912.0f;
}

// stage the voltages of batch g (Q frames of one channel) into vs[FB][row_pitch]
template <int Q, int NT>
__device__ __forceinline__ void stage_voltages(const FusedParams& P, uint8_t* vs, int c, int b, int tid) {
  const size_t frame_stride = (size_t)P.n_chan * P.row_bytes;
  const uint8_t* src0 = P.volt + (size_t)c * P.row_bytes;
  if (P.aligned16) {
    const int chunks = P.row_pitch >> 4;
    for (int i = tid; i < Q * chunks; i += NT) {
      const int f = i / chunks, k = i - f * chunks;
      const int t = b * Q + f;
      uint8_t* dst = vs + f * P.row_pitch + k * 16;
      if (t < P.n_t) cp_async16(dst, src0 + (size_t)t * frame_stride + k * 16);
      else *reinterpret_cast<uint4*>(dst) = make_uint4(0u, 0u, 0u, 0u);
    }
  } else {
    for (int i = tid; i < Q * P.row_bytes; i += NT) {
      const int f = i / P.row_bytes, k = i - f * P.row_bytes;
      const int t = b * Q + f;
      vs[f * P.row_pitch + k] = (t < P.n_t) ? src0[(size_t)t * frame_stride + k] : (uint8_t)0;
    }
  }
  cp_async_commit();
}

// S1 + S3 for the batch: every thread owns the block cells tid + j*NT and sums their gather
// lists, in table order, for all Q*NPOL (frame, pol) planes.  A zero byte is the zero sample.
template <int Q, int NPOL, int NT, bool DELTA>
__device__ __forceinline__ void gather_batch(const FusedParams& P, const uint8_t* __restrict__ vs,
                                             float2* __restrict__ gh, const uint32_t (&info)[S * S / NT],
                                             int tid) {
  constexpr int PL = Q * NPOL;
#pragma unroll
  for (int j = 0; j < S * S / NT; ++j) {
    const int cell = tid + j * NT;
    const int cy = cell >> 5, cx = cell & 31;
    if (cy >= P.R) continue;
    const uint32_t beg = info[j] >> 8, cnt = info[j] & 0xFFu;
    float2* dst = gh + cy * HS + cx;
    if (DELTA) {
      uint32_t s[PL];
#pragma unroll
      for (int pl = 0; pl < PL; ++pl) s[pl] = 0u;
      for (uint32_t e = beg; e < beg + cnt; ++e) {
        const int a = __ldg(P.ent_ant + e);
#pragma unroll
        for (int pl = 0; pl < PL; ++pl) {
          const int f = pl / NPOL, pol = pl % NPOL;
          s[pl] += unpack_biased(vs[f * P.row_pitch + pol * P.n_ant + a]);
        }
      }
      const int bias = 8 * (int)cnt;
#pragma unroll
      for (int pl = 0; pl < PL; ++pl) {
        const float re = small_int_to_float((int)(s[pl] >> 16) - bias);
        const float im = small_int_to_float((int)(s[pl] & 0xFFFFu) - bias);
        dst[pl * (S * HS)] = make_float2(re, im);
      }
    } else {
      float2 s[PL];
#pragma unroll
      for (int pl = 0; pl < PL; ++pl) s[pl] = make_float2(0.0f, 0.0f);
      for (uint32_t e = beg; e < beg + cnt; ++e) {
        const int a = __ldg(P.ent_ant + e);
        const float2 w = __ldg(P.ent_tap + e);
#pragma unroll
        for (int pl = 0; pl < PL; ++pl) {
          const int f = pl / NPOL, pol = pl % NPOL;
          const uint32_t u = unpack_biased(vs[f * P.row_pitch + pol * P.n_ant + a]);
          const float er = small_int_to_float((int)(u >> 16) - 8);
          const float ei = small_int_to_float((int)(u & 0xFFFFu) - 8);
          s[pl].x = fmaf(w.x, er, s[pl].x); s[pl].x = fmaf(-w.y, ei, s[pl].x);
          s[pl].y = fmaf(w.x, ei, s[pl].y); s[pl].y = fmaf(w.y, er, s[pl].y);
        }
      }
#pragma unroll
      for (int pl = 0; pl < PL; ++pl) dst[pl * (S * HS)] = s[pl];
    }
  }
}

// rows: thread = (frame f, pol, row y); in place on its own row of gh[f][pol]
template <int Q, int RHO>
__device__ __forceinline__ void row_task(float2* __restrict__ row, int n_valid) {
  C2 z[16];
  dft32_pair<Q, RHO>(z, row, 1, n_valid);
  // output k: lo -> l1 = 2k, hi -> l1 = 2k+1 (l = Q l1 + l2): one 16-byte store per k
  float4* out = reinterpret_cast<float4*>(row);
#pragma unroll
  for (int k = 0; k < 16; ++k) out[k] = make_float4(z[k].re.x, z[k].im.x, z[k].re.y, z[k].im.y);
}

// columns + S5 + S6: thread = (pol, m2 = RHO, l1); acc[k] = (m = 2Q k + RHO, m = 2Q k + RHO + Q)
template <int Q, int RHO>
__device__ __forceinline__ void col_task_power(const float2* __restrict__ col, int n_valid, float2 (&acc)[16]) {
  C2 z[16];
  dft32_pair<Q, RHO>(z, col, HS, n_valid);
#pragma unroll
  for (int k = 0; k < 16; ++k) {
    acc[k] = __ffma2_rn(z[k].re, z[k].re, acc[k]);
    acc[k] = __ffma2_rn(z[k].im, z[k].im, acc[k]);
  }
}

template <int Q, int R0>
__device__ __forceinline__ void row_dispatch(int rho, float2* row, int n_valid) {
  if constexpr (R0 < Q) {
    if (rho == R0) row_task<Q, R0>(row, n_valid);
    else row_dispatch<Q, R0 + 1>(rho, row, n_valid);
  }
}
template <int Q, int R0>
__device__ __forceinline__ void col_dispatch(int rho, const float2* col, int n_valid, float2 (&acc)[16]) {
  if constexpr (R0 < Q) {
    if (rho == R0) col_task_power<Q, R0>(col, n_valid, acc);
    else col_dispatch<Q, R0 + 1>(rho, col, n_valid, acc);
  }
}

template <int Q, int NPOL>
struct FusedGeo {
  static constexpr int NT = NPOL * Q * 32;                 // threads per CTA
  static constexpr int PLANE = S * HS;                     // complex elements per (frame, pol) plane
  static constexpr size_t GH_BYTES = (size_t)Q * NPOL * PLANE * sizeof(float2);
};

template <int Q, int NPOL, bool DELTA>
__global__ void __launch_bounds__(NPOL * Q * 32, (NPOL * Q * 32 <= 256) ? 2 : 1)
epic_fused_kernel(FusedParams P) {
  using G = FusedGeo<Q, NPOL>;
  constexpr int NT = G::NT, N = 32 * Q;
  extern __shared__ __align__(16) unsigned char smem_raw[];
  float2* gh = reinterpret_cast<float2*>(smem_raw);        // [Q][NPOL][32][HS]
  uint8_t* vs = smem_raw + G::GH_BYTES;                    // [2][Q][row_pitch]
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;

  // static, contiguous share of the (unit-major, batch-minor) work list
  const long long g0 = P.total * (long long)blockIdx.x / gridDim.x;
  const long long g1 = P.total * (long long)(blockIdx.x + 1) / gridDim.x;
  if (g0 >= g1) return;

  uint32_t info[S * S / NT];
#pragma unroll
  for (int j = 0; j < S * S / NT; ++j) info[j] = __ldg(P.cell_info + tid + j * NT);

  // column-stage role: warp -> m2, lanes -> (pol, l1)
  const int m2 = warp / NPOL;
  const int pol_c = (NPOL == 2) ? (lane >> 4) : 0;
  const int l1 = (NPOL == 2) ? ((warp & 1) * 16 + (lane & 15)) : lane;
  // row-stage role: warp -> (frame, pol), lane -> row
  const int f_r = warp / NPOL, pol_r = warp % NPOL;

  float2 acc[16];
#pragma unroll
  for (int k = 0; k < 16; ++k) acc[k] = make_float2(0.0f, 0.0f);

  auto flush = [&](int unit) {
    const int c = unit / Q, l2 = unit - c * Q;
    float* o = P.out + ((size_t)c * P.n_planes + pol_c) * (size_t)(N * N) + (Q * l1 + l2);
#pragma unroll
    for (int k = 0; k < 16; ++k) {
      atomicAdd(o + (size_t)(2 * Q * k + m2) * N, acc[k].x);
      atomicAdd(o + (size_t)(2 * Q * k + m2 + Q) * N, acc[k].y);
      acc[k] = make_float2(0.0f, 0.0f);
    }
  };

  int unit = (int)(g0 / P.nb);
  int b = (int)(g0 - (long long)unit * P.nb);
  int buf = 0;
  stage_voltages<Q, NT>(P, vs, unit / Q, b, tid);
  for (long long g = g0; g < g1; ++g) {
    cp_async_wait_all();
    __syncthreads();  // this batch's voltages are visible; previous column stage is done with gh
    // prefetch the next batch
    int unit_n = unit, b_n = b + 1;
    if (b_n == P.nb) { b_n = 0; ++unit_n; }
    if (g + 1 < g1) stage_voltages<Q, NT>(P, vs + (buf ^ 1) * Q * P.row_pitch, unit_n / Q, b_n, tid);

    gather_batch<Q, NPOL, NT, DELTA>(P, vs + buf * Q * P.row_pitch, gh, info, tid);
    __syncthreads();
    if (lane < P.R) row_dispatch<Q, 0>(unit % Q, gh + (f_r * NPOL + pol_r) * G::PLANE + lane * HS, P.Cc);
    __syncthreads();
#pragma unroll 1
    for (int f = 0; f < Q; ++f)
      col_dispatch<Q, 0>(m2, gh + (f * NPOL + pol_c) * G::PLANE + l1, P.R, acc);

    if (unit_n != unit || g + 1 == g1) flush(unit);
    unit = unit_n; b = b_n; buf ^= 1;
  }
}

struct FusedTables {
  uint32_t* cell_info;
};

template <int Q, int NPOL, bool DELTA>
int launch_fused(const epic_plan* p, const FusedParams& P, cudaStream_t s) {
  using G = FusedGeo<Q, NPOL>;
  const size_t smem = G::GH_BYTES + (size_t)2 * Q * P.row_pitch;
  auto kern = epic_fused_kernel<Q, NPOL, DELTA>;
  if (smem > 48 * 1024)
    EPIC_CUDA_TRY(cudaFuncSetAttribute((const void*)kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
  int per_sm = 0;
  EPIC_CUDA_TRY(cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, kern, G::NT, smem));
  if (per_sm < 1) return EPIC_ERR_RANGE;
  const long long slots = (long long)per_sm * p->n_sm;
  const int grid = (int)std::min<long long>(P.total, slots);
  kern<<<grid, G::NT, smem, s>>>(P);
  EPIC_CUDA_TRY(cudaGetLastError());
  return EPIC_OK;
}

template <int Q>
int launch_fused_q(const epic_plan* p, const FusedParams& P, int n_pol, cudaStream_t s) {
  const bool delta = p->t.is_delta != 0;
  if (n_pol == 1) return delta ? launch_fused<Q, 1, true>(p, P, s) : launch_fused<Q, 1, false>(p, P, s);
  return delta ? launch_fused<Q, 2, true>(p, P, s) : launch_fused<Q, 2, false>(p, P, s);
}

}  // namespace

// ---------------------------------------------------------------- host side
int fused_plan_init(epic_plan* p) {
  p->fused_ok = 0;
  p->d_fused = nullptr;
  const int Q = p->N / S;
  if (p->N % S != 0 || (Q != 2 && Q != 4)) return EPIC_OK;
  if (p->R > S || p->Cc > S) return EPIC_OK;
  if (p->h_ent_ant.size() >= ((size_t)1 << 24)) return EPIC_OK;
  std::vector<uint32_t> info((size_t)S * S, 0u);
  for (const CellRec& c : p->h_cells) {
    if (c.ent_count > 255u) return EPIC_OK;  // falls back to the two-pass path
    info[(size_t)c.y * S + c.x] = (c.ent_begin << 8) | c.ent_count;
  }
  FusedTables* ft = new (std::nothrow) FusedTables();
  if (!ft) return EPIC_ERR_NOMEM;
  ft->cell_info = nullptr;
  cudaError_t ce = cudaMalloc(&ft->cell_info, info.size() * sizeof(uint32_t));
  if (ce == cudaSuccess)
    ce = cudaMemcpy(ft->cell_info, info.data(), info.size() * sizeof(uint32_t), cudaMemcpyHostToDevice);
  if (ce != cudaSuccess) {
    set_cuda_error(ce);
    if (ft->cell_info) cudaFree(ft->cell_info);
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
    delete ft;
  }
  p->d_fused = nullptr;
  p->fused_ok = 0;
}

int fused_supported(const epic_plan* p, int is_cf32, int n_pol, int n_products) {
  if (!p->fused_ok || is_cf32) return 0;
  if (n_products != n_pol) return 0;  // {XX} or {XX, YY}
  const size_t pitch = ((size_t)n_pol * p->n_ant + 15) & ~(size_t)15;
  const int Q = p->N / S;
  const size_t smem = (size_t)Q * n_pol * S * HS * sizeof(float2) + 2 * Q * pitch;
  return smem <= (size_t)200 * 1024 ? 1 : 0;
}

int fused_image(epic_plan* p, const ImageArgs& a) {
  const FusedTables* ft = static_cast<const FusedTables*>(p->d_fused);
  const int Q = p->N / S;
  FusedParams P;
  P.volt = static_cast<const uint8_t*>(a.volt);
  P.out = a.out;
  P.cell_info = ft->cell_info;
  P.ent_ant = p->t.ent_ant;
  P.ent_tap = p->t.ent_tap;
  P.n_t = a.n_t;
  P.n_chan = a.n_chan;
  P.n_ant = p->n_ant;
  P.n_planes = a.n_planes;
  P.R = p->R;
  P.Cc = p->Cc;
  P.nb = (a.n_t + Q - 1) / Q;
  P.total = (long long)a.n_chan * Q * P.nb;
  P.row_bytes = a.n_pol * p->n_ant;
  P.row_pitch = (P.row_bytes + 15) & ~15;
  P.aligned16 = (P.row_bytes % 16 == 0 && (reinterpret_cast<uintptr_t>(a.volt) & 15u) == 0) ? 1 : 0;
  int st;
  if (Q == 2) st = launch_fused_q<2>(p, P, a.n_pol, a.stream);
  else st = launch_fused_q<4>(p, P, a.n_pol, a.stream);
  if (st != EPIC_OK) return st;
  p->last_launches = 1;
  return EPIC_OK;
}

}  // namespace epic
