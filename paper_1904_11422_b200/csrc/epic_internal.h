// Internal declarations shared by the libepic.so translation units (not part of the ABI).
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>
#include <vector>

#include "epic.h"

namespace epic {

// One nonzero cell of the (relocated) support block and its gather list (S2 inverted:
// per-cell list of (antenna, tap) pairs, built once on the host).
struct CellRec {
  uint16_t y, x;      // relocated coordinates inside the support box
  uint32_t ent_begin; // first entry in ent_ant / ent_tap
  uint32_t ent_count;
};

struct DevTables {
  // With n_layout > 1 (one antenna layout per channel, reading Q15) the tables of the
  // layouts are concatenated: channel c's row pointers start at row_ptr + c * row_stride and hold
  // indices into the common cells array, whose ent_begin index the common entry arrays.
  const CellRec* cells;     // [n_cells], each layout's cells sorted by (y, x)
  const uint32_t* row_ptr;  // [n_layout][R + 1]: cells of support row y are [row_ptr[y], row_ptr[y+1])
  const uint16_t* ent_ant;  // [n_ent] antenna index of each gather entry
  const float2* ent_tap;    // [n_ent] complex tap of each gather entry
  const float2* twiddle;    // [N/2]: exp(+2 pi i k / N), computed in double on the host
  int n_cells, n_ent;
  int N, logN, R, Cc, y0, x0; // support box: rows [y0, y0+R) mod N, cols [x0, x0+Cc) mod N
  int n_ant, is_delta;
  int n_layout, row_stride; // row_stride = R + 1 when n_layout > 1, else 0 (every channel reads layout 0)
};

} // namespace epic

namespace epic {
// epic_image_host: double-buffered device staging of the voltages, a device copy of out_accum, two streams
struct HostPipe {
  cudaStream_t compute, copy, back;  // kernels; host->device copies; device->host copies of finished channel chunks
  cudaEvent_t copied[2], consumed[2];
  void* d_volt[2];
  size_t volt_bytes;   // capacity of each staging buffer
  float* d_out;
  size_t out_bytes;    // capacity of d_out
};
}  // namespace epic

struct epic_plan {
  int grid_n, pad, N, logN, n_ant, K;
  int n_products_req; // 0 = default
  int path_req;
  int last_launches;
  int n_layout;                // antenna layouts: 1, or one per channel
  std::vector<int> cells_host; // [n_layout][n_ant][K][K] true cells y*N + x
  int y0, x0, R, Cc;
  epic::DevTables t;           // device pointers
  void* d_blob;                // one allocation holding all tables
  void* d_scratch;             // two-pass intermediate H, L2-sized
  size_t scratch_bytes;
  size_t scratch_limit;        // bytes of the scratch a batch may use (0 = all of it)
  void* d_fused;               // tables private to the fused path
  int fused_ok;                // support fits the fused kernel
  void* d_tiled;               // tables private to the tiled path
  void* d_wide;                // tables private to the wide fused path (support within 64 x 64)
  int wide_ok;                 // support fits the wide fused kernel (and not the 32 x 32 one)
  void* d_auto;                // tap autocorrelation table of epic_autocorr_remove
  int input_order;             // EPIC_ORDER_TCPA | EPIC_ORDER_TCAP
  int ph_n_chan, ph_n_pol;     // shape of the delay phasor table (0: none set)
  float2* d_phasor;            // [ph_n_chan][ph_n_pol][n_ant] complex multipliers (reading Q19)
  float4* d_phasor_pair;       // [ph_n_chan][n_ant] (re_lo, re_hi, im_lo, im_hi): lo/hi = pol X/Y, or the same pol twice
  int tiled_ok;                // N is 256 or 512
  epic::HostPipe* pipe;        // streams, events and device staging of epic_image_host (created on first use)
  int n_sm;
  // host copies kept for the fused path's table builder
  std::vector<epic::CellRec> h_cells;   // all layouts, concatenated
  std::vector<uint32_t> h_cell_off;     // [n_layout + 1]: layout l's cells are [h_cell_off[l], h_cell_off[l+1])
  std::vector<uint16_t> h_ent_ant;
  std::vector<float2> h_ent_tap;
  std::vector<uint16_t> h_slot_order;   // tap plans that fit 32x32: per layout, the fused kernel's slot list as
                                        // cells y*32+x of the R x 32 block (bank_order_entries); else empty
};

namespace epic {

struct ImageArgs {
  const void* volt;
  int is_cf32;
  int native;                  // voltages in [T][C][A][Np] order (else [T][C][Np][A])
  const float2* phasor;        // delay phasors [C][Np][A] or nullptr
  const float4* phasor_pair;   // the same, pair-packed [C][A], or nullptr
  int n_t, n_chan, n_pol, n_products, n_planes;
  float* out;
  cudaStream_t stream;
};

// epic_twopass.cu
int twopass_image(epic_plan* p, const ImageArgs& a);
int debug_grid(epic_plan* p, int layout, const void* volt, int is_cf32, int n_pol, float* out, cudaStream_t s);
int debug_unpack(const void* bytes, long n, float* out, cudaStream_t s);
int fp32_probe(int iters, float* ms, double* flops);

// epic_fused.cu
int fused_plan_init(epic_plan* p);  // sets p->fused_ok, allocates p->d_fused
void fused_plan_free(epic_plan* p);
int fused_supported(const epic_plan* p, int is_cf32, int n_pol, int n_products);
int fused_image(epic_plan* p, const ImageArgs& a);
int fused_image_noalloc(epic_plan* p, const ImageArgs& a);  // the residue-group kernel with the static scratch array
long long noalloc_scratch_bytes();
int tensor_supported(const epic_plan* p, int is_cf32, int n_pol, int n_products);  // tensor-core column pass
int tensor_image(epic_plan* p, const ImageArgs& a);

// epic_wide.cu: the fused design for supports up to 64 x 64 (reached through EPIC_PATH_FUSED)
int wide_plan_init(epic_plan* p);  // sets p->wide_ok, allocates p->d_wide
void wide_plan_free(epic_plan* p);
int wide_supported(const epic_plan* p, int is_cf32, int n_pol, int n_products);
int wide_image(epic_plan* p, const ImageArgs& a);

// epic_tiled.cu
int tiled_plan_init(epic_plan* p);  // sets p->tiled_ok, allocates p->d_tiled
void tiled_plan_free(epic_plan* p);
int tiled_supported(const epic_plan* p, int is_cf32, int n_pol, int n_products);
int tiled_image(epic_plan* p, const ImageArgs& a);
int stream_supported(const epic_plan* p, int is_cf32, int n_pol, int n_products);  // persistent producer/consumer variant
int stream_image(epic_plan* p, const ImageArgs& a);

// epic_autocorr.cu
int autocorr_plan_init(epic_plan* p, const float* taps);  // allocates p->d_auto
void autocorr_plan_free(epic_plan* p);
int autocorr_remove(epic_plan* p, const ImageArgs& a);

void set_cuda_error(cudaError_t e);

// bytes of the plan's scratch one batch may use
inline size_t scratch_budget(const epic_plan* p) {
  return (p->scratch_limit != 0 && p->scratch_limit < p->scratch_bytes) ? p->scratch_limit : p->scratch_bytes;
}

} // namespace epic

#define EPIC_CUDA_TRY(expr)                         \
  do {                                              \
    cudaError_t e__ = (expr);                       \
    if (e__ != cudaSuccess) {                       \
      epic::set_cuda_error(e__);                    \
      return EPIC_ERR_CUDA;                         \
    }                                               \
  } while (0)
