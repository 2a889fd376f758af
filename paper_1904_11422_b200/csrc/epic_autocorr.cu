// Optional autocorrelation removal ("autocorrelation removal can also be done to
// remove the zero-spacing power inherent in EPIC").  The accumulated EPIC image is the direct-
// Fourier image of ALL antenna pairs, a = b included (DESIGN.md check (a)):
//
//   I_pq[m][l] = sum_t A_p A_q^*,  A_p[m][l] = sum_a E_ap(t) What_a[m][l],
//   What_a[m][l] = sum_d W_a[d] exp(+2 pi i ((cx_a + dx) l + (cy_a + dy) m) / N)
//
// and its a = b part is  sum_a V_aa^pq |What_a[m][l]|^2  with V_aa^pq = sum_t E_ap E_aq^*.
// |What_a|^2 does not depend on the antenna's cell, only on its taps:
//   |What_a|^2 = sum_lag corr_a[lag] exp(+2 pi i (lag_x l + lag_y m) / N),
//   corr_a[lag] = sum_d W_a[d] conj(W_a[d - lag]),  lag in [-(K-1), K-1]^2   (plan table, from double).
//
//   kernel 1  autocorr_power     V_aa^pq per (channel, time chunk, antenna), exact integer sums
//   kernel 2  autocorr_sum       chunk sums, in order
//   kernel 3  autocorr_lags      L_pq[c][lag] = sum_a V_aa^pq corr_a[lag]
//   kernel 4  autocorr_subtract  out_accum[c][plane][m][l] -= sum_lag L_pq[c][lag] W_N^{lag_x l + lag_y m}
//
// HBM-bound and small next to epic_image (the voltages are read once more); no atomics.
#include <algorithm>
#include <cmath>
#include <new>
#include <vector>

#include "epic_internal.h"

namespace epic {
namespace {

constexpr int CHUNKS = 16;  // time chunks of kernel 1 (parallelism); summed in order by kernel 2

__device__ __forceinline__ int sext4_hi(uint32_t b) { return ((int)(int8_t)(b & 0xFFu)) >> 4; }
__device__ __forceinline__ int sext4_lo(uint32_t b) { return ((int)(int8_t)((b << 4) & 0xFFu)) >> 4; }

// power[(c * CHUNKS + chunk) * A + a] = (sum |E_x|^2, sum |E_y|^2, Re sum E_x E_y^*, Im sum E_x E_y^*)
// One thread follows VEC consecutive antennas (VEC = 4: aligned 32-bit loads) through the chunk's samples.
template <int VEC>
__global__ void __launch_bounds__(128) autocorr_power(const uint8_t* __restrict__ volt, int n_t, int n_chan,
                                                      int n_pol, int n_ant, int native, int4* __restrict__ power) {
  const int chunk = blockIdx.x, c = blockIdx.y;
  const int t0 = (int)((long long)n_t * chunk / CHUNKS), t1 = (int)((long long)n_t * (chunk + 1) / CHUNKS);
  const size_t row = (size_t)n_pol * n_ant, step = (size_t)n_chan * row;
  for (int a = VEC * (blockIdx.z * blockDim.x + threadIdx.x); a < n_ant; a += VEC * blockDim.x * gridDim.z) {
    int xx[VEC], yy[VEC], xyr[VEC], xyi[VEC];
#pragma unroll
    for (int i = 0; i < VEC; ++i) xx[i] = yy[i] = xyr[i] = xyi[i] = 0;
    const bool tcap = native && n_pol == 2;  // untransposed order: (a X, a Y) byte pairs
    const uint8_t* p = volt + ((size_t)t0 * n_chan + c) * row + (tcap ? 2 * a : a);
    for (int t = t0; t < t1; ++t, p += step) {
      uint32_t wx, wy = 0u;
      if (tcap) {
        if (VEC == 4) {
          const uint32_t w0 = __ldg(reinterpret_cast<const uint32_t*>(p)), w1 = __ldg(reinterpret_cast<const uint32_t*>(p) + 1);
          wx = __byte_perm(w0, w1, 0x6420u);
          wy = __byte_perm(w0, w1, 0x7531u);
        } else {
          wx = __ldg(p);
          wy = __ldg(p + 1);
        }
      } else if (VEC == 4) {
        wx = __ldg(reinterpret_cast<const uint32_t*>(p));
        if (n_pol == 2) wy = __ldg(reinterpret_cast<const uint32_t*>(p + n_ant));
      } else {
        wx = __ldg(p);
        if (n_pol == 2) wy = __ldg(p + n_ant);
      }
#pragma unroll
      for (int i = 0; i < VEC; ++i) {
        const uint32_t bx = (wx >> (8 * i)) & 0xFFu, by = (wy >> (8 * i)) & 0xFFu;
        const int xr = sext4_hi(bx), xi = sext4_lo(bx), yr = sext4_hi(by), yi = sext4_lo(by);
        xx[i] += xr * xr + xi * xi;
        yy[i] += yr * yr + yi * yi;
        xyr[i] += xr * yr + xi * yi;  // E_x conj(E_y) (reading Q11)
        xyi[i] += xi * yr - xr * yi;
      }
    }
#pragma unroll
    for (int i = 0; i < VEC; ++i)
      power[((size_t)c * CHUNKS + chunk) * n_ant + a + i] = make_int4(xx[i], yy[i], xyr[i], xyi[i]);
  }
}

// psum[c * A + a] = chunk-summed power as floats (the integer sums are exact; the order is fixed)
// With delay phasors d (reading Q19) the compensated powers are |d_x|^2 xx, |d_y|^2 yy, d_x conj(d_y) xy.
__global__ void __launch_bounds__(256) autocorr_sum(const int4* __restrict__ power, int n_chan, int n_ant,
                                                    const float4* __restrict__ phasor, float4* __restrict__ psum) {
  const int i = blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= n_chan * n_ant) return;
  const int c = i / n_ant, a = i - c * n_ant;
  int xx = 0, yy = 0, xyr = 0, xyi = 0;
#pragma unroll
  for (int k = 0; k < CHUNKS; ++k) {
    const int4 v = __ldg(power + ((size_t)c * CHUNKS + k) * n_ant + a);
    xx += v.x; yy += v.y; xyr += v.z; xyi += v.w;
  }
  float4 v = make_float4((float)xx, (float)yy, (float)xyr, (float)xyi);
  if (phasor) {
    const float4 d = __ldg(phasor + i);  // (re_x, re_y, im_x, im_y)
    const float gr = d.x * d.y + d.z * d.w, gi = d.z * d.y - d.x * d.w;  // d_x conj(d_y)
    v = make_float4(v.x * (d.x * d.x + d.z * d.z), v.y * (d.y * d.y + d.w * d.w), v.z * gr - v.w * gi, v.z * gi + v.w * gr);
  }
  psum[i] = v;
}

// lags[(c * n_lag + q) * 6] = (Lxx.re, Lxx.im, Lyy.re, Lyy.im, Lxy.re, Lxy.im) = sum_a V_aa corr_a[q].
// One warp per (channel, lag): lanes stride the antennas, then a fixed shuffle tree (deterministic).
__global__ void __launch_bounds__(128) autocorr_lags(const float4* __restrict__ psum, const float2* __restrict__ corr,
                                                     int n_ant, int n_lag, int corr_stride, float* __restrict__ lags) {
  const int c = blockIdx.x, q = blockIdx.y * 4 + (threadIdx.x >> 5), lane = threadIdx.x & 31;
  if (q >= n_lag) return;
  corr += (size_t)c * corr_stride * n_lag;  // this channel's layout (corr_stride = 0: one layout)
  float v[6] = {0.f, 0.f, 0.f, 0.f, 0.f, 0.f};
  for (int a = lane; a < n_ant; a += 32) {
    const float4 p = __ldg(psum + (size_t)c * n_ant + a);
    const float2 w = __ldg(corr + (size_t)a * n_lag + q);
    v[0] = fmaf(p.x, w.x, v[0]); v[1] = fmaf(p.x, w.y, v[1]);
    v[2] = fmaf(p.y, w.x, v[2]); v[3] = fmaf(p.y, w.y, v[3]);
    v[4] = fmaf(p.z, w.x, v[4]); v[4] = fmaf(-p.w, w.y, v[4]);
    v[5] = fmaf(p.z, w.y, v[5]); v[5] = fmaf(p.w, w.x, v[5]);
  }
#pragma unroll
  for (int off = 16; off > 0; off >>= 1)
#pragma unroll
    for (int k = 0; k < 6; ++k) v[k] += __shfl_xor_sync(0xFFFFFFFFu, v[k], off);
  if (lane == 0) {
    float* o = lags + ((size_t)c * n_lag + q) * 6;
#pragma unroll
    for (int k = 0; k < 6; ++k) o[k] = v[k];
  }
}

__global__ void __launch_bounds__(256) autocorr_subtract(const float* __restrict__ lags, const float2* __restrict__ tw,
                                                         int N, int K, int n_planes, float* __restrict__ out) {
  const int c = blockIdx.y;
  const int px = blockIdx.x * blockDim.x + threadIdx.x;
  if (px >= N * N) return;
  const int m = px / N, l = px - m * N;
  const int span = 2 * K - 1, n_lag = span * span;
  float xx = 0.f, yy = 0.f, xyr = 0.f, xyi = 0.f;
  for (int q = 0; q < n_lag; ++q) {
    const int ly = q / span - (K - 1), lx = q % span - (K - 1);
    const int k = (lx * l + ly * m) & (N - 1);  // N is a power of two; & is the positive modulus
    float2 w = __ldg(tw + (k & (N / 2 - 1)));   // exp(+2 pi i k / N), table holds k < N/2
    if (k >= N / 2) { w.x = -w.x; w.y = -w.y; }
    const float* L = lags + ((size_t)c * n_lag + q) * 6;
    xx += L[0] * w.x - L[1] * w.y;
    yy += L[2] * w.x - L[3] * w.y;
    xyr += L[4] * w.x - L[5] * w.y;
    xyi += L[4] * w.y + L[5] * w.x;
  }
  const size_t plane = (size_t)N * N;
  float* o = out + (size_t)c * n_planes * plane + px;
  o[0] -= xx;
  if (n_planes >= 2) o[plane] -= yy;
  if (n_planes == 6) {  // YX = conj(XY)
    o[2 * plane] -= xyr;
    o[3 * plane] -= xyi;
    o[4 * plane] -= xyr;
    o[5 * plane] += xyi;
  }
}

struct AutoTables {
  float2* corr;  // [n_layout][A][(2K-1)^2]
};

}  // namespace

int autocorr_plan_init(epic_plan* p, const float* taps) {
  p->d_auto = nullptr;
  const int K = p->K, span = 2 * K - 1, n_lag = span * span, A = p->n_ant * p->n_layout;  // (layout, antenna) rows
  std::vector<float2> corr((size_t)A * n_lag);
  for (int a = 0; a < A; ++a)
    for (int ly = -(K - 1); ly <= K - 1; ++ly)
      for (int lx = -(K - 1); lx <= K - 1; ++lx) {
        double re = 0.0, im = 0.0;
        for (int dy = 0; dy < K; ++dy)
          for (int dx = 0; dx < K; ++dx) {
            const int ey = dy - ly, ex = dx - lx;  // d' = d - lag
            if (ey < 0 || ey >= K || ex < 0 || ex >= K) continue;
            double wr = 1.0, wi = 0.0, vr = 1.0, vi = 0.0;
            if (taps) {
              wr = taps[(((size_t)a * K + dy) * K + dx) * 2]; wi = taps[(((size_t)a * K + dy) * K + dx) * 2 + 1];
              vr = taps[(((size_t)a * K + ey) * K + ex) * 2]; vi = taps[(((size_t)a * K + ey) * K + ex) * 2 + 1];
            }
            re += wr * vr + wi * vi;  // W[d] conj(W[d'])
            im += wi * vr - wr * vi;
          }
        corr[(size_t)a * n_lag + (size_t)(ly + K - 1) * span + (lx + K - 1)] = make_float2((float)re, (float)im);
      }
  AutoTables* at = new (std::nothrow) AutoTables();
  if (!at) return EPIC_ERR_NOMEM;
  at->corr = nullptr;
  cudaError_t ce = cudaMalloc(&at->corr, corr.size() * sizeof(float2));
  if (ce == cudaSuccess) ce = cudaMemcpy(at->corr, corr.data(), corr.size() * sizeof(float2), cudaMemcpyHostToDevice);
  if (ce != cudaSuccess) {
    set_cuda_error(ce);
    if (at->corr) cudaFree(at->corr);
    delete at;
    return ce == cudaErrorMemoryAllocation ? EPIC_ERR_NOMEM : EPIC_ERR_CUDA;
  }
  p->d_auto = at;
  return EPIC_OK;
}

void autocorr_plan_free(epic_plan* p) {
  AutoTables* at = static_cast<AutoTables*>(p->d_auto);
  if (at) {
    if (at->corr) cudaFree(at->corr);
    delete at;
  }
  p->d_auto = nullptr;
}

int autocorr_remove(epic_plan* p, const ImageArgs& a) {
  const AutoTables* at = static_cast<const AutoTables*>(p->d_auto);
  const int K = p->K, n_lag = (2 * K - 1) * (2 * K - 1), A = p->n_ant, N = p->N;
  const size_t power_bytes = (size_t)a.n_chan * CHUNKS * A * sizeof(int4);
  const size_t psum_bytes = (size_t)a.n_chan * A * sizeof(float4);
  const size_t lag_bytes = (size_t)a.n_chan * n_lag * 6 * sizeof(float);
  if (power_bytes + psum_bytes + lag_bytes > p->scratch_bytes) return EPIC_ERR_RANGE;
  int4* power = static_cast<int4*>(p->d_scratch);
  float4* psum = reinterpret_cast<float4*>(static_cast<char*>(p->d_scratch) + power_bytes);
  float* lags = reinterpret_cast<float*>(static_cast<char*>(p->d_scratch) + power_bytes + psum_bytes);
  const uint8_t* volt = static_cast<const uint8_t*>(a.volt);
  if (A % 4 == 0 && (reinterpret_cast<uintptr_t>(volt) & 3u) == 0) {
    const int gz = std::max(1, std::min(8, A / 4 / 128));
    autocorr_power<4><<<dim3(CHUNKS, a.n_chan, gz), 128, 0, a.stream>>>(volt, a.n_t, a.n_chan, a.n_pol, A, a.native, power);
  } else {
    const int gz = std::max(1, std::min(8, A / 128));
    autocorr_power<1><<<dim3(CHUNKS, a.n_chan, gz), 128, 0, a.stream>>>(volt, a.n_t, a.n_chan, a.n_pol, A, a.native, power);
  }
  autocorr_sum<<<(a.n_chan * A + 255) / 256, 256, 0, a.stream>>>(power, a.n_chan, A, a.phasor_pair, psum);
  autocorr_lags<<<dim3(a.n_chan, (n_lag + 3) / 4), 128, 0, a.stream>>>(psum, at->corr, A, n_lag,
                                                                         p->n_layout > 1 ? A : 0, lags);
  autocorr_subtract<<<dim3((N * N + 255) / 256, a.n_chan), 256, 0, a.stream>>>(lags, p->t.twiddle, N, K, a.n_planes,
                                                                              a.out);
  EPIC_CUDA_TRY(cudaGetLastError());
  p->last_launches = 4;
  return EPIC_OK;
}

}  // namespace epic
