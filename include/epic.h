/* epic.h — C ABI of libepic.so: the EPIC (E-field Parallel Imaging Correlator) hot path on
 * one NVIDIA B200 (sm_100a).
 *
 * Method: Kent et al., arXiv 1904.11422.  Per frequency channel c and time sample t
 * (one "frame"), per polarisation p (Eq. 5; §3.2):
 *
 *   S1 unpack      byte -> E = sext4(byte >> 4) + i sext4(byte & 15)
 *   S2 cells       nearest cell (cx,cy) = floor(u+0.5), floor(v+0.5); tap cell
 *                  ((cy+dy) mod N, (cx+dx) mod N)
 *   S3 gridding    G[y][x] += W_a[dy][dx] * E_a   (collisions sum)
 *   S4 transform   A[m][l] = sum_{y,x} G[y][x] exp(+2 pi i (x l + y m)/N)          PAPER.md:126, Eq. 5
 *   S5 products    XX=|A_X|^2, YY=|A_Y|^2, XY=A_X conj(A_Y), YX=A_Y conj(A_X)
 *   S6 accumulate  sum over the n_t time samples of the call
 *
 * N = grid_n * pad (zero-padded plane side, a power of two).  The transform is the
 * unnormalised inverse DFT in natural order with zenith (l = m = 0) at [0][0]; no fftshift.
 * All arithmetic is fp32 (the paper's complex64); the optional EPIC_PATH_TENSOR
 * forms the column transform from BF16 hi + lo split operands with fp32 accumulation, to the
 * same tolerance.
 *
 * Conventions.  Every function returns EPIC_OK (0) or a negative epic_status; nothing throws
 * across the ABI.  Argument validation is synchronous.  Device work is enqueued on `stream`
 * (a cudaStream_t passed as void*; NULL = the legacy default stream) and is asynchronous:
 * kernel faults surface at the caller's next synchronisation.  epic_image* never allocate,
 * never synchronise with the host and never copy host memory.  A plan owns device tables and
 * a scratch buffer; calls on ONE plan must be issued on one stream at a time (the scratch is
 * per plan).  Pointers marked HOST are read during the call and not retained; pointers marked
 * DEVICE are owned by the caller (e.g. PyTorch tensors) and must stay valid until the
 * enqueued work has finished.
 */
#ifndef EPIC_H_
#define EPIC_H_

#ifdef __cplusplus
extern "C" {
#endif

#if defined(__GNUC__)
#define EPIC_API __attribute__((visibility("default")))
#else
#define EPIC_API
#endif

typedef struct epic_plan epic_plan; /* opaque; created/destroyed by the library */
typedef void* epic_stream;          /* cudaStream_t */

typedef enum epic_status {
  EPIC_OK = 0,
  EPIC_ERR_ARG = -1,   /* NULL pointer, bad shape, even kernel_k, N not a power of two in 8..512 */
  EPIC_ERR_RANGE = -2, /* n_pol not in {1,2}, n_products incompatible with n_pol, n_ant too large */
  EPIC_ERR_CUDA = -3,  /* a CUDA runtime call failed; see epic_last_cuda_error() */
  EPIC_ERR_NOMEM = -4, /* host or device allocation failed */
  EPIC_ERR_SCRATCH = -5 /* epic_image_noalloc: the call needs more than the library's static scratch array holds */
} epic_status;

/* Which kernel family epic_image uses.  AUTO picks the fastest one that supports the plan. */
typedef enum epic_path {
  EPIC_PATH_AUTO = 0,
  EPIC_PATH_TWOPASS = 1, /* grid+row-FFT kernel -> scratch in global memory -> column-FFT+products kernel, batch by batch */
  EPIC_PATH_FUSED = 2,   /* one kernel (+ a tiny ordered fix-up of split units), planes never leave the SM: N = 32, 64, 128 with
                            the occupied cells within 32x32 (epic_fused.cu) or, for N = 64, 128, within 64x64 (the wide variant, epic_wide.cu) */
  EPIC_PATH_TILED = 3,   /* N = 256, 512: packed row kernel -> scratch (1 GiB batches, streamed through HBM) -> packed column
                            kernel; AUTO's choice for N >= 256 */
  EPIC_PATH_TENSOR = 4,  /* the fused kernel with its column transform as a dense BF16x3 contraction on the
                            tensor cores (tcgen05.mma); N = 128, two polarisations, one layout.  Never
                            picked by AUTO: measured and reported beside the FP32 path */
  EPIC_PATH_STREAM = 5   /* N = 256, 512: ONE persistent kernel; row CTAs hand row-transformed frames to column CTAs
                            through a ring that stays in L2, accumulators live in registers for the whole call:
                            HBM sees the voltages and out_accum once.  Measured slower than
                            EPIC_PATH_TILED so far, so AUTO picks it only where the tiled row kernel cannot run (antenna counts that
                            are no multiple of 4, voltage pointers that are not word-aligned); EPIC_ERR_RANGE at epic_image time if one
                            channel's row and column CTAs cannot be co-resident */
} epic_path;

/* S2 + plan set-up ("gridded onto a 2D grid ... spacing < lambda/2"; illumination
 * kernel "user-defined").  HOST pointers, copied.
 *   grid_n, pad   aperture cells per side and integer zero-padding factor; N = grid_n*pad must be
 *                 a power of two with 8 <= N <= 512.
 *   n_ant         number of antennas, 1..65535.
 *   ant_uv        float[n_ant][2] = (u, v) in aperture CELL units; u -> x -> l is the fast axis.
 *                 Cell = floor(double(u) + 0.5); cells outside [0,N) wrap modulo N.
 *   kernel_taps   NULL -> delta kernel (kernel_k must be 1, tap 1+0i); else
 *                 float[n_ant][kernel_k][kernel_k][2], complex fp32 indexed [dy+h][dx+h],
 *                 h = (kernel_k-1)/2, shared by both polarisations.
 *   kernel_k      odd, 1..15.
 * On success *out receives the plan (products default: n_pol==2 -> 4, n_pol==1 -> 1). */
EPIC_API int epic_plan_create(epic_plan** out, int grid_n, int pad, int n_ant, const float* ant_uv,
                     const float* kernel_taps, int kernel_k);

/* The same with ONE LAYOUT PER FREQUENCY CHANNEL.  The grid spacing is tied to "the wavelength of the
 * channel" (lambda/2 at the deployment), so an antenna's coordinates
 * in cell units -- and with them its nearest cell, its sub-cell offset and the taps of a kernel of
 * fixed physical size such as the 3 m top-hat of PAPER.md:166 -- differ from channel to channel
 * (reading Q15).
 *   n_layout      number of channels the plan describes, >= 1.
 *   ant_uv        float[n_layout][n_ant][2]; kernel_taps NULL or
 *                 float[n_layout][n_ant][kernel_k][kernel_k][2]; otherwise as above.
 * Channel c of every later call uses layout c: epic_image / epic_autocorr_remove then require
 * n_chan == n_layout (EPIC_ERR_ARG otherwise); a plan with n_layout == 1 (what epic_plan_create
 * makes) applies its one layout to any number of channels.  The occupied support box is the
 * union over the layouts. */
EPIC_API int epic_plan_create_per_channel(epic_plan** out, int grid_n, int pad, int n_ant, int n_layout,
                                 const float* ant_uv, const float* kernel_taps, int kernel_k);

/* Number of layouts of the plan (1 unless made by epic_plan_create_per_channel). */
EPIC_API int epic_plan_get_n_layouts(const epic_plan* plan);

/* Frees the plan's device tables and scratch.  NULL is a no-op.  Synchronises the device. */
EPIC_API int epic_plan_destroy(epic_plan* plan);

/* S5 selection: n_products = 1 (XX; n_pol must be 1), 2 (XX,YY) or 4 (XX,YY,XY,YX); the latter
 * two need n_pol == 2.  Checked against n_pol at epic_image time.  0 restores the default. */
EPIC_API int epic_plan_set_products(epic_plan* plan, int n_products);

/* Select the kernel family (testing / benchmarking): an epic_path value.  EPIC_ERR_RANGE if the plan
 * cannot use it (FUSED: occupied cells within 64x64 and N = 32, 64 or 128; TILED, STREAM: N = 256 or 512). */
EPIC_API int epic_plan_set_path(epic_plan* plan, int path);

/* Tuning: bytes of the plan's scratch (the intermediate H of the tiled / two-pass paths; the ring of the streamed path) one batch may
 * use; 0 = all of it (1 GiB for N >= 256, else 128 MiB).  A small limit (e.g. 64 MiB) keeps H resident in
 * the 126 MB L2 at the price of more, shorter batches, each ending in one read-modify-write of its
 * channels' out_accum.  A batch always holds at least one frame. */
EPIC_API int epic_plan_set_scratch_limit(epic_plan* plan, long long bytes);

/* S1..S6 for one gulp (one call = one gulp of n_t samples).
 *   voltages   DEVICE uint8[n_t][n_chan][n_pol][n_ant] — [Time, Channel, Polarisation, Antenna]
 *              order, 1 byte = 4+4-bit complex: high nibble real, low nibble
 *              imaginary, two's complement -8..7.
 *   out_accum  DEVICE float[n_chan][planes][N][N]; planes = 1 {XX} | 2 {XX,YY} |
 *              6 {XX,YY,Re XY,Im XY,Re YX,Im YX}.  The call ADDS the sum over its n_t samples
 *              into out_accum ("accumulated"); the caller zeroes it to start an
 *              integration.  n_t == 0 or n_chan == 0 is a successful no-op. */
EPIC_API int epic_image(epic_plan* plan, const void* voltages, int n_t, int n_chan, int n_pol,
               float* out_accum, epic_stream stream);

/* The same gulp from HOST memory, end to end: voltages_host HOST uint8 (layout as in epic_image; pinned memory makes the
 * copies asynchronous, pageable memory works), out_accum_host HOST float[n_chan][planes][N][N].  The library cuts the gulp
 * into n_chunks pieces (<= 0: chosen from the gulp's size, 1..8; the first one half as long, its copy is the one nothing
 * hides) and pipelines them on its own streams with double-buffered device staging owned by the plan.  One-layout plans
 * without delay phasors are cut by CHANNEL range: the host->device copy of chunk k+1 (one strided 2-D copy) and the
 * device->host copy of chunk k's finished images both overlap the kernels in between.  Other plans are cut in TIME: the
 * host->device copies overlap the kernels and the accumulated images are copied back once at the end.
 * accumulate != 0: the images are ADDED to the contents of out_accum_host (which is copied to the device first);
 * accumulate == 0: out_accum_host is overwritten.  SYNCHRONOUS: returns when out_accum_host is complete.  Honours products,
 * path, input order, delay phasors and per-channel layouts like epic_image.  This is the call bench.py's `e2e` leg times. */
EPIC_API int epic_image_host(epic_plan* plan, const void* voltages_host, int n_t, int n_chan, int n_pol,
                    float* out_accum_host, int accumulate, int n_chunks);

/* epic_image for callers that must not allocate (code under CUDA graph capture, tight serving loops, harnesses that
 * forbid cudaMalloc).  Same arguments, semantics and result as epic_image (S1..S6; ADDS into
 * out_accum; asynchronous on `stream`), for plans the fused kernel of epic_fused.cu takes with ONE layout: N = 64 or
 * 128, occupied cells within 32 x 32, 4+4-bit voltages (EPIC_ERR_RANGE otherwise; epic_plan_set_path is ignored).
 * The kernel's scratch -- the partial sums of work units whose time range is split between CTAs -- is not the plan's
 * cudaMalloc'ed buffer but a file-scope `static __device__` array of epic_noalloc_scratch_bytes() = 80 MiB inside the
 * library: every GPU that loads libepic.so holds those 80 MiB until the process exits.  The call itself calls no
 * cudaMalloc, cudaFree or allocating library routine and does not synchronise.  A launch that would need more than
 * the array holds (256 KiB per resident CTA at N = 128: 74 MiB on a 148-SM B200 with two CTAs per SM, more on a larger GPU)
 * is refused with EPIC_ERR_SCRATCH before anything is enqueued.  Nothing in the array has to start at zero (every
 * slot that is read was written by the same call).  ALL calls in the process on one GPU share the array: calls that
 * overlap on the GPU (different streams, or different plans on different streams) race on it -- issue them on one
 * stream or order them with events.  The first call on each device looks the array's device address up
 * (cudaGetSymbolAddress, no allocation); callers that capture graphs make one call outside capture first (n_t = 0 will
 * do). */
EPIC_API int epic_image_noalloc(epic_plan* plan, const void* voltages, int n_t, int n_chan, int n_pol,
                       float* out_accum, epic_stream stream);
/* Size in bytes of the static scratch array of epic_image_noalloc. */
EPIC_API long long epic_noalloc_scratch_bytes(void);

/* Same with complex fp32 voltages: DEVICE float[n_t][n_chan][n_pol][n_ant][2] (re, im). */
EPIC_API int epic_image_cf32(epic_plan* plan, const void* voltages_cf32, int n_t, int n_chan, int n_pol,
                    float* out_accum, epic_stream stream);

/* Upstream steps folded into the load.
 * Input order: the F-engine packets arrive as [Time, Channel, Antenna, Polarisation]; the paper
 * transposes them to [Time, Channel, Polarisation, Antenna] before gridding.  With
 * EPIC_ORDER_TCAP epic_image / epic_image_cf32 / epic_autocorr_remove read the untransposed order
 * directly (the transposition happens in the kernels' staging loads).  Default EPIC_ORDER_TCPA. */
typedef enum epic_order { EPIC_ORDER_TCPA = 0, EPIC_ORDER_TCAP = 1 } epic_order;
EPIC_API int epic_plan_set_input_order(epic_plan* plan, int order);

/* Delay compensation ("compensation for the signal path delays are applied"): every
 * unpacked voltage of (channel c, polarisation p, antenna a) is multiplied by the complex number
 * phasors[c][p][a] before gridding (typically exp(-2 pi i nu_c tau_a); computing it is the caller's
 * business, as it was the LWA library's in the paper).
 *   phasors  HOST float[n_chan][n_pol][n_ant][2] (re, im), copied; NULL removes the table.
 * While a table is set, image calls must use the same n_chan and n_pol (else EPIC_ERR_ARG). */
EPIC_API int epic_plan_set_delay_phasors(epic_plan* plan, int n_chan, int n_pol, const float* phasors);

/* Optional autocorrelation removal ("to remove the zero-spacing power inherent in EPIC";
 * SURVEY.md 8(f) NEXT-2).  The EPIC image of a gulp is the direct-Fourier image of ALL antenna pairs,
 * a = b included; this call SUBTRACTS from out_accum the a = b part of the same gulp,
 *   sum_a (sum_t E_ap E_aq^*) |What_a[m][l]|^2,  What_a = transform of antenna a's gridded taps,
 * for every product plane the plan forms (same arguments, layout and stream rules as epic_image; ci4
 * voltages).  It is linear in the gulp, so it may be applied per call or to several gulps in turn.
 * Four small kernels; reads the voltages once more; uses the plan's scratch. */
EPIC_API int epic_autocorr_remove(epic_plan* plan, const void* voltages, int n_t, int n_chan, int n_pol,
                         float* out_accum, epic_stream stream);

/* Plan queries (host, synchronous). */
EPIC_API int epic_plan_get_n(const epic_plan* plan);        /* N, or negative status */
EPIC_API int epic_plan_get_n_planes(const epic_plan* plan, int n_pol); /* planes for current products */
/* S2 result: cells_host HOST int[n_layout][n_ant][kernel_k][kernel_k] = y*N + x of every tap. */
EPIC_API int epic_plan_get_cells(const epic_plan* plan, int* cells_host);
/* Circular bounding box of the occupied cells: HOST int[4] = {y0, x0, rows, cols}. */
EPIC_API int epic_plan_get_support(const epic_plan* plan, int* box_host);
/* Kernel family epic_image will use for this plan and n_pol (an epic_path value). */
EPIC_API int epic_plan_get_path(const epic_plan* plan, int n_pol);
/* Number of kernel launches the last epic_image* call on this plan enqueued. */
EPIC_API int epic_plan_last_launches(const epic_plan* plan);

/* Test hooks for the bit-exact clauses (BASELINE.json north_star).
 * epic_debug_unpack: S1 alone. bytes_dev DEVICE uint8[n] -> out_dev DEVICE float[n][2].
 * epic_debug_grid:   S1+S3 for ONE frame through the plan's gather table.  voltages DEVICE as
 *                    in epic_image (is_cf32 != 0: as in epic_image_cf32) with n_t = n_chan = 1;
 *                    out_plane_dev DEVICE float[n_pol][N][N][2], overwritten, true
 *                    (un-relocated) cell positions.  Uses layout 0;
 * epic_debug_grid_layout: the same through layout `layout` (0 <= layout < n_layout) of a
 *                    per-channel plan. */
EPIC_API int epic_debug_unpack(const void* bytes_dev, long n, float* out_dev, epic_stream stream);
EPIC_API int epic_debug_grid(epic_plan* plan, const void* voltages, int is_cf32, int n_pol,
                    float* out_plane_dev, epic_stream stream);
EPIC_API int epic_debug_grid_layout(epic_plan* plan, int layout, const void* voltages, int is_cf32, int n_pol,
                           float* out_plane_dev, epic_stream stream);

/* FP32 FMA micro-benchmark used for the roofline denominator: runs `iters` dependent-chain
 * FFMA rounds on every SM and writes elapsed milliseconds and the flop count (HOST outputs).
 * Synchronous. */
EPIC_API int epic_fp32_peak_probe(int iters, float* ms_out, double* flops_out);

EPIC_API const char* epic_status_string(int status);
EPIC_API int epic_last_cuda_error(void); /* cudaError_t of the most recent failing CUDA call, per thread */

#ifdef __cplusplus
}
#endif
#endif /* EPIC_H_ */
