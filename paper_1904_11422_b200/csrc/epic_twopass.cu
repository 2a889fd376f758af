// General EPIC path for any plan (N = 8..512, any support, 1 or 2 polarisations, ci4 or cf32):
//
//   kernel A  grid_rowfft   S1 unpack + S3 gather-gridding of a chunk of support rows into shared
//                           memory, S4 along x (row transforms), rows written to the scratch H
//   kernel B  colfft_accum  S4 along y for a strip of image columns, S5 products, S6 accumulation
//                           over the time samples of the batch in registers, one add into out_accum
//
// H (complex fp32 [frame][pol][R][N], only the R occupied rows) lives in an L2-sized scratch, so
// HBM sees the voltages once and out_accum once per batch.  Only the R x Cc support box of the
// aperture plane is ever formed: the box is relocated to the origin, which multiplies both
// polarisations' images by the same unit-modulus phase ramp and cancels in every product
// (SURVEY.md reading Q7).  Transforms are radix-2 Stockham passes in shared memory (natural
// order in and out) with the plan's double-precision-derived twiddle table.
#include <algorithm>

#include "epic_internal.h"

namespace epic {

// ---------------------------------------------------------------- S1: 4+4-bit unpack
// PAPER.md:120-122; reading Q1: high nibble real, low nibble imaginary, two's complement.
__device__ __forceinline__ float2 unpack_ci4(uint32_t b) {
  const int re = ((int)(int8_t)(b & 0xFFu)) >> 4;
  const int im = ((int)(int8_t)((b << 4) & 0xFFu)) >> 4;
  return make_float2((float)re, (float)im);
}

__device__ __forceinline__ float2 cmul(float2 a, float2 w) {
  return make_float2(fmaf(a.x, w.x, -a.y * w.y), fmaf(a.x, w.y, a.y * w.x));
}

// ---------------------------------------------------------------- S3: one cell of the gather
// G[cell] = sum over the cell's (antenna, tap) list of W * E, in (antenna, tap) order
// (PAPER.md:122-124).  v points at this frame-and-polarisation's antenna vector.
// Antenna a's sample is v[a * a_stride] (a_stride = n_pol for the untransposed input order,
// PAPER.md:120); `ph` (or nullptr) holds this channel-and-polarisation's delay phasors
// (reading Q19).
template <bool CF32>
__device__ __forceinline__ float2 gather_cell(const DevTables& t, const CellRec c, const void* v, int a_stride = 1,
                                              const float2* __restrict__ ph = nullptr) {
  float2 s = make_float2(0.0f, 0.0f);
  for (uint32_t e = c.ent_begin; e < c.ent_begin + c.ent_count; ++e) {
    const int a = t.ent_ant[e];
    const float2 w = t.ent_tap[e];
    float2 E;
    if (CF32) E = reinterpret_cast<const float2*>(v)[(size_t)a * a_stride];
    else E = unpack_ci4(reinterpret_cast<const uint8_t*>(v)[(size_t)a * a_stride]);
    if (ph) E = cmul(E, ph[a]);
    s.x = fmaf(w.x, E.x, s.x);
    s.x = fmaf(-w.y, E.y, s.x);
    s.y = fmaf(w.x, E.y, s.y);
    s.y = fmaf(w.y, E.x, s.y);
  }
  return s;
}

// One radix-2 Stockham pass over `n_seq` sequences of length N stored with stride `seq_stride`:
// y[2(j-k)+k] = x[j] + w x[j+N/2], y[2(j-k)+k+s] = x[j] - w x[j+N/2], k = j mod s,
// w = exp(+2 pi i k/(2s)).  After log2 N passes (s = 1, 2, .., N/2) the result is the
// unnormalised inverse DFT in natural order (Eq. 5; readings Q8-Q10).
__device__ __forceinline__ void stockham_pass(const float2* __restrict__ x, float2* __restrict__ y,
                                              const float2* __restrict__ tw, int n_seq,
                                              int seq_stride, int N, int logN, int s, int log_s,
                                              int tid, int n_thr) {
  const int half = N >> 1;
  const int total = n_seq << (logN - 1);
  for (int i = tid; i < total; i += n_thr) {
    const int q = i >> (logN - 1);
    const int j = i & (half - 1);
    const int k = j & (s - 1);
    const float2 w = tw[k << (logN - 1 - log_s)];
    const float2* xs = x + q * seq_stride;
    float2* ys = y + q * seq_stride;
    const float2 a = xs[j];
    const float2 b = cmul(xs[j + half], w);
    const int o = ((j - k) << 1) + k;
    ys[o] = make_float2(a.x + b.x, a.y + b.y);
    ys[o + s] = make_float2(a.x - b.x, a.y - b.y);
  }
}

struct BatchGeom {
  int c0, t0, Cb, Tb; // batch = channels [c0, c0+Cb) x times [t0, t0+Tb)
  int C, Np, A;       // call shape
  int RB;             // support rows per kernel-A block
  int W;              // image columns per kernel-B block
  int native;         // input order [T][C][A][Np] instead of [T][C][Np][A]
  const float2* phasor; // delay phasors [C][Np][A] or nullptr
};

// ---------------------------------------------------------------- kernel A
template <bool CF32>
__global__ void __launch_bounds__(256) grid_rowfft(DevTables t, BatchGeom g, const void* volt,
                                                   float2* __restrict__ H) {
  extern __shared__ float2 sm[];
  const int N = t.N, logN = t.logN;
  float2* tw = sm;                 // [N/2]
  float2* bx = sm + (N >> 1);      // [RB][N]
  float2* by = bx + g.RB * N;      // [RB][N]
  const int tid = threadIdx.x;
  const int pol = blockIdx.y;
  const int fb = blockIdx.z;       // frame in batch: cb * Tb + tb
  const int cb = fb / g.Tb, tb = fb - cb * g.Tb;
  const int r0 = blockIdx.x * g.RB;
  const int rows = min(g.RB, t.R - r0);
  const size_t vidx = ((size_t)(g.t0 + tb) * g.C + (g.c0 + cb)) * g.Np * (size_t)g.A +
                      (g.native ? (size_t)pol : (size_t)pol * g.A);
  const int a_stride = g.native ? g.Np : 1;
  const float2* ph = g.phasor ? g.phasor + ((size_t)(g.c0 + cb) * g.Np + pol) * g.A : nullptr;
  const void* v = CF32 ? (const void*)(reinterpret_cast<const float2*>(volt) + vidx)
                       : (const void*)(reinterpret_cast<const uint8_t*>(volt) + vidx);
  for (int i = tid; i < (N >> 1); i += 256) tw[i] = t.twiddle[i];
  for (int i = tid; i < rows * N; i += 256) bx[i] = make_float2(0.0f, 0.0f);
  __syncthreads();
  const uint32_t* rp = t.row_ptr + (size_t)(g.c0 + cb) * t.row_stride;  // this channel's layout
  const uint32_t cbeg = rp[r0], cend = rp[r0 + rows];
  for (uint32_t ci = cbeg + tid; ci < cend; ci += 256) {
    const CellRec c = t.cells[ci];
    bx[(c.y - r0) * N + c.x] = gather_cell<CF32>(t, c, v, a_stride, ph);
  }
  __syncthreads();
  float2* x = bx;
  float2* y = by;
  for (int ls = 0; ls < logN; ++ls) {
    stockham_pass(x, y, tw, rows, N, N, logN, 1 << ls, ls, tid, 256);
    __syncthreads();
    float2* tmp = x; x = y; y = tmp;
  }
  float2* dst = H + (((size_t)fb * g.Np + pol) * t.R + r0) * (size_t)N;
  for (int i = tid; i < rows * N; i += 256) dst[i] = x[i];
}

// ---------------------------------------------------------------- kernel B
// PIX = pixels per thread = W*N/256 (<= 8).
template <int NPOL, int NPROD>
__global__ void __launch_bounds__(256) colfft_accum(DevTables t, BatchGeom g,
                                                    const float2* __restrict__ H,
                                                    float* __restrict__ out, int n_planes) {
  extern __shared__ float2 sm[];
  constexpr int NACC = (NPROD == 4) ? 4 : NPOL;
  constexpr int MAXPIX = 8;
  const int N = t.N, logN = t.logN, W = g.W;
  const int NS = N + 1;            // padded column stride (complex elements)
  float2* tw = sm;                 // [N/2]
  float2* bx = sm + (N >> 1);      // [NPOL][W][NS]
  float2* by = bx + NPOL * W * NS;
  const int tid = threadIdx.x;
  const int strip = blockIdx.x;
  const int cb = blockIdx.y;
  const int l0 = strip * W;
  const int npix = W * N;          // per polarisation
  float acc[MAXPIX][NACC];
#pragma unroll
  for (int q = 0; q < MAXPIX; ++q)
#pragma unroll
    for (int k = 0; k < NACC; ++k) acc[q][k] = 0.0f;
  for (int i = tid; i < (N >> 1); i += 256) tw[i] = t.twiddle[i];

  for (int tb = 0; tb < g.Tb; ++tb) {
    const int fb = cb * g.Tb + tb;
    __syncthreads(); // previous frame's products are done with bx/by
    // load the strip of H, transposed to [col][n]; rows n >= R are structurally zero
    for (int p = 0; p < NPOL; ++p) {
      const float2* src = H + ((size_t)fb * NPOL + p) * t.R * (size_t)N + l0;
      float2* dstp = bx + p * W * NS;
      for (int i = tid; i < npix; i += 256) {
        const int col = i % W, n = i / W;
        dstp[col * NS + n] = (n < t.R) ? src[(size_t)n * N + col] : make_float2(0.0f, 0.0f);
      }
    }
    __syncthreads();
    float2* x = bx;
    float2* y = by;
    for (int ls = 0; ls < logN; ++ls) {
      stockham_pass(x, y, tw, NPOL * W, NS, N, logN, 1 << ls, ls, tid, 256);
      __syncthreads();
      float2* tmp = x; x = y; y = tmp;
    }
    // S5 + S6: pixel i -> (col = i % W, m = i / W)
#pragma unroll
    for (int q = 0; q < MAXPIX; ++q) {
      const int i = tid + q * 256;
      if (i < npix) {
        const int col = i % W, m = i / W;
        const float2 ax = x[col * NS + m];
        acc[q][0] = fmaf(ax.x, ax.x, fmaf(ax.y, ax.y, acc[q][0]));
        if (NPOL == 2) {
          const float2 ay = x[(W + col) * NS + m];
          acc[q][1] = fmaf(ay.x, ay.x, fmaf(ay.y, ay.y, acc[q][1]));
          if (NPROD == 4) { // XY = A_X conj(A_Y) (reading Q11, Eq. 2)
            acc[q][2] = fmaf(ax.x, ay.x, fmaf(ax.y, ay.y, acc[q][2]));
            acc[q][3] = fmaf(ax.y, ay.x, fmaf(-ax.x, ay.y, acc[q][3]));
          }
        }
      }
    }
  }
  // one add into out_accum per batch; this block is the only writer of its (channel, strip)
  float* o = out + (size_t)(g.c0 + cb) * n_planes * N * (size_t)N;
  const size_t plane = (size_t)N * N;
#pragma unroll
  for (int q = 0; q < MAXPIX; ++q) {
    const int i = tid + q * 256;
    if (i < npix) {
      const int col = i % W, m = i / W;
      const size_t px = (size_t)m * N + l0 + col;
      o[px] += acc[q][0];
      if (NPOL == 2) {
        o[plane + px] += acc[q][1];
        if (NPROD == 4) { // YX = conj(XY)
          o[2 * plane + px] += acc[q][2];
          o[3 * plane + px] += acc[q][3];
          o[4 * plane + px] += acc[q][2];
          o[5 * plane + px] -= acc[q][3];
        }
      }
    }
  }
}

static int set_smem(const void* fn, size_t bytes) {
  if (bytes > 48 * 1024)
    EPIC_CUDA_TRY(cudaFuncSetAttribute(fn, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)bytes));
  return EPIC_OK;
}

template <int NPOL, int NPROD>
static int launch_colfft(const epic_plan* p, const BatchGeom& g, int strips, size_t smem,
                         const ImageArgs& a) {
  int st = set_smem((const void*)colfft_accum<NPOL, NPROD>, smem);
  if (st != EPIC_OK) return st;
  colfft_accum<NPOL, NPROD><<<dim3(strips, g.Cb), 256, smem, a.stream>>>(
      p->t, g, (const float2*)p->d_scratch, a.out, a.n_planes);
  return EPIC_OK;
}

int twopass_image(epic_plan* p, const ImageArgs& a) {
  const int N = p->N, R = p->R;
  BatchGeom g;
  g.C = a.n_chan;
  g.Np = a.n_pol;
  g.A = p->n_ant;
  g.native = a.native;
  g.phasor = a.phasor;
  g.RB = std::max(1, std::min(R, 2048 / N));
  g.W = std::max(1, std::min(N, 2048 / N));
  const int strips = N / g.W;
  const size_t frame_bytes = (size_t)a.n_pol * R * N * sizeof(float2);
  const long long max_frames = (long long)std::max<size_t>(1, scratch_budget(p) / frame_bytes);
  const int want_blocks = 2 * p->n_sm;
  long long Cb = std::min<long long>(a.n_chan, (want_blocks + strips - 1) / strips);
  Cb = std::max<long long>(1, std::min(Cb, max_frames));
  long long Tb = std::max<long long>(1, std::min<long long>(a.n_t, max_frames / Cb));
  // gridDim.z limit of kernel A
  while (Cb * Tb > 65535) { if (Tb > 1) Tb = (Tb + 1) / 2; else Cb = (Cb + 1) / 2; }
  const size_t smem_a = ((size_t)(N / 2) + 2 * (size_t)g.RB * N) * sizeof(float2);
  const size_t smem_b = ((size_t)(N / 2) + 2 * (size_t)a.n_pol * g.W * (N + 1)) * sizeof(float2);
  int st = a.is_cf32 ? set_smem((const void*)grid_rowfft<true>, smem_a)
                     : set_smem((const void*)grid_rowfft<false>, smem_a);
  if (st != EPIC_OK) return st;
  const int chunks = (R + g.RB - 1) / g.RB;
  int launches = 0;
  for (int c0 = 0; c0 < a.n_chan; c0 += (int)Cb) {
    g.c0 = c0;
    g.Cb = (int)std::min<long long>(Cb, a.n_chan - c0);
    for (int t0 = 0; t0 < a.n_t; t0 += (int)Tb) {
      g.t0 = t0;
      g.Tb = (int)std::min<long long>(Tb, a.n_t - t0);
      const dim3 grid_a(chunks, a.n_pol, g.Cb * g.Tb);
      if (a.is_cf32)
        grid_rowfft<true><<<grid_a, 256, smem_a, a.stream>>>(p->t, g, a.volt, (float2*)p->d_scratch);
      else
        grid_rowfft<false><<<grid_a, 256, smem_a, a.stream>>>(p->t, g, a.volt, (float2*)p->d_scratch);
      if (a.n_pol == 1) st = launch_colfft<1, 1>(p, g, strips, smem_b, a);
      else if (a.n_products == 2) st = launch_colfft<2, 2>(p, g, strips, smem_b, a);
      else st = launch_colfft<2, 4>(p, g, strips, smem_b, a);
      if (st != EPIC_OK) return st;
      launches += 2;
    }
  }
  EPIC_CUDA_TRY(cudaGetLastError());
  p->last_launches = launches;
  return EPIC_OK;
}

// ---------------------------------------------------------------- test hooks
__global__ void unpack_kernel(const uint8_t* __restrict__ b, long n, float2* __restrict__ out) {
  for (long i = blockIdx.x * (long)blockDim.x + threadIdx.x; i < n; i += (long)gridDim.x * blockDim.x)
    out[i] = unpack_ci4(b[i]);
}

int debug_unpack(const void* bytes, long n, float* out, cudaStream_t s) {
  const int blocks = (int)std::min<long>(1184, (n + 255) / 256);
  unpack_kernel<<<blocks, 256, 0, s>>>((const uint8_t*)bytes, n, (float2*)out);
  EPIC_CUDA_TRY(cudaGetLastError());
  return EPIC_OK;
}

template <bool CF32>
__global__ void grid_plane_kernel(DevTables t, int layout, const void* volt, int n_pol, float2* __restrict__ out) {
  const int pol = blockIdx.y;
  const uint32_t* rp = t.row_ptr + (size_t)layout * (t.R + 1);
  const int c_begin = rp[0], c_end = rp[t.R];
  const void* v = CF32 ? (const void*)(reinterpret_cast<const float2*>(volt) + (size_t)pol * t.n_ant)
                       : (const void*)(reinterpret_cast<const uint8_t*>(volt) + (size_t)pol * t.n_ant);
  for (int ci = c_begin + blockIdx.x * blockDim.x + threadIdx.x; ci < c_end; ci += gridDim.x * blockDim.x) {
    const CellRec c = t.cells[ci];
    const int y = (c.y + t.y0) & (t.N - 1), x = (c.x + t.x0) & (t.N - 1);
    out[((size_t)pol * t.N + y) * t.N + x] = gather_cell<CF32>(t, c, v);
  }
}

int debug_grid(epic_plan* p, int layout, const void* volt, int is_cf32, int n_pol, float* out, cudaStream_t s) {
  EPIC_CUDA_TRY(cudaMemsetAsync(out, 0, (size_t)n_pol * p->N * p->N * sizeof(float2), s));
  const int n_cells = (int)(p->h_cell_off[layout + 1] - p->h_cell_off[layout]);
  const dim3 grid((n_cells + 255) / 256, n_pol);
  if (is_cf32) grid_plane_kernel<true><<<grid, 256, 0, s>>>(p->t, layout, volt, n_pol, (float2*)out);
  else grid_plane_kernel<false><<<grid, 256, 0, s>>>(p->t, layout, volt, n_pol, (float2*)out);
  EPIC_CUDA_TRY(cudaGetLastError());
  return EPIC_OK;
}

// ---------------------------------------------------------------- FP32 FMA probe (roofline denominator)
// 8 independent FFMA chains per thread, 64 FFMA per loop trip.
__global__ void __launch_bounds__(256) fma_probe_kernel(int iters, float seed, float* sink) {
  float a0 = seed + threadIdx.x, a1 = a0 + 1.f, a2 = a0 + 2.f, a3 = a0 + 3.f;
  float a4 = a0 + 4.f, a5 = a0 + 5.f, a6 = a0 + 6.f, a7 = a0 + 7.f;
  const float m = 0.999f + seed, c = 0.001f;
  for (int i = 0; i < iters; ++i) {
#pragma unroll
    for (int u = 0; u < 8; ++u) {
      a0 = fmaf(a0, m, c); a1 = fmaf(a1, m, c); a2 = fmaf(a2, m, c); a3 = fmaf(a3, m, c);
      a4 = fmaf(a4, m, c); a5 = fmaf(a5, m, c); a6 = fmaf(a6, m, c); a7 = fmaf(a7, m, c);
    }
  }
  const float r = ((a0 + a1) + (a2 + a3)) + ((a4 + a5) + (a6 + a7));
  if (r == 12345.678f) sink[0] = r;
}

int fp32_probe(int iters, float* ms, double* flops) {
  int dev = 0, n_sm = 0;
  EPIC_CUDA_TRY(cudaGetDevice(&dev));
  EPIC_CUDA_TRY(cudaDeviceGetAttribute(&n_sm, cudaDevAttrMultiProcessorCount, dev));
  float* sink = nullptr;
  EPIC_CUDA_TRY(cudaMalloc(&sink, sizeof(float)));
  cudaEvent_t e0, e1;
  EPIC_CUDA_TRY(cudaEventCreate(&e0));
  EPIC_CUDA_TRY(cudaEventCreate(&e1));
  const int blocks = n_sm * 8;
  fma_probe_kernel<<<blocks, 256>>>(iters / 8 + 1, 0.0f, sink); // warm-up
  EPIC_CUDA_TRY(cudaEventRecord(e0));
  fma_probe_kernel<<<blocks, 256>>>(iters, 0.0f, sink);
  EPIC_CUDA_TRY(cudaEventRecord(e1));
  EPIC_CUDA_TRY(cudaEventSynchronize(e1));
  EPIC_CUDA_TRY(cudaEventElapsedTime(ms, e0, e1));
  *flops = (double)blocks * 256.0 * 64.0 * 2.0 * (double)iters;
  cudaEventDestroy(e0);
  cudaEventDestroy(e1);
  cudaFree(sink);
  return EPIC_OK;
}

} // namespace epic
