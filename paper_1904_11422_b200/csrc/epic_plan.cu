// libepic.so — host side: plan construction (S2: cell indexing) and the C ABI
// declared in include/epic.h.  No arithmetic of the per-frame path lives here; the kernels are
// in epic_twopass.cu (general two-kernel path) and epic_fused.cu (one-kernel path).
#include <algorithm>
#include <cmath>
#include <cstring>
#include <new>

#include "epic_internal.h"

namespace epic {

static thread_local int g_last_cuda_error = 0;
void set_cuda_error(cudaError_t e) { g_last_cuda_error = (int)e; }

static inline int pos_mod(long long v, int n) {
  long long m = v % n;
  return (int)(m < 0 ? m + n : m);
}

// Smallest circular interval [start, start+len) mod n that covers every index with occ[i] != 0.
static void circular_box(const std::vector<char>& occ, int n, int* start, int* len) {
  int n_occ = 0;
  for (int i = 0; i < n; ++i) n_occ += occ[i] ? 1 : 0;
  if (n_occ == 0) { *start = 0; *len = 1; return; }
  // longest run of empty indices on the circle
  int best_len = 0, best_end = 0; // run occupies (best_end - best_len, best_end]  (indices mod n)
  int run = 0;
  for (int i = 0; i < 2 * n; ++i) {
    if (!occ[i % n]) {
      ++run;
      if (run > best_len && run <= n) { best_len = run; best_end = i % n; }
    } else {
      run = 0;
    }
  }
  if (best_len >= n) { *start = 0; *len = 1; return; }
  *start = (best_end + 1) % n;
  *len = n - best_len;
}

struct Entry {
  int y, x;      // relocated
  int ant, tap;  // tap = iy*K + ix
};

// Slot order and entry order for the fused kernel's gather (epic_fused.cu, gather_batch): a
// quarter-warp owns 8 consecutive cells of the slot list (descending entry count, so that warps
// see uniform trip counts) and step i of its loop reads entry i of each cell with one LDS.128 of
// E[antenna]; that load is conflict-free when the 8 antennas differ mod 8 (16-byte bank groups)
// or coincide (broadcast).  Two greedy passes at plan time: (1) among the next cells of equal
// count, a group takes the one whose antennas share the fewest bank groups (and the most
// antennas) with the group so far; (2) per group and step, each cell takes the remaining entry
// whose bank group holds the fewest other antennas so far.  Only the order of a cell's sum
// changes (rounding order; PAPER.md:122-124 fixes none).  Appends the layout's R*32 slots to
// h_slot_order.
static void bank_order_entries(epic_plan* p, size_t cell0) {
  constexpr int S = 32, G = 8, WINDOW = 96;
  std::vector<const CellRec*> dense((size_t)S * S, nullptr);
  for (size_t i = cell0; i < p->h_cells.size(); ++i) {
    const CellRec& c = p->h_cells[i];
    dense[(size_t)c.y * S + c.x] = &c;
  }
  auto count_of = [&](uint16_t s) { return dense[s] ? dense[s]->ent_count : 0u; };
  std::vector<uint16_t> rest;  // descending count, stable in (y, x)
  for (int y = 0; y < p->R; ++y)
    for (int x = 0; x < S; ++x) rest.push_back((uint16_t)(y * S + x));
  std::stable_sort(rest.begin(), rest.end(), [&](uint16_t a, uint16_t b) { return count_of(a) > count_of(b); });
  // (1) groups of G slots
  std::vector<uint16_t> order;
  order.reserve(rest.size());
  size_t head = 0;
  std::vector<char> taken(rest.size(), 0);
  while (order.size() < rest.size()) {
    std::vector<uint16_t> grp_ants;
    for (int lane = 0; lane < G && order.size() < rest.size(); ++lane) {
      while (taken[head]) ++head;
      const uint32_t cnt = count_of(rest[head]);
      size_t pick = head;
      if (cnt > 0 && !grp_ants.empty()) {
        long best = 0;
        bool have = false;
        size_t seen = 0;
        for (size_t i = head; i < rest.size() && seen < WINDOW; ++i) {
          if (taken[i]) continue;
          if (count_of(rest[i]) != cnt) break;
          ++seen;
          const CellRec* c = dense[rest[i]];
          long cost = 0;
          for (uint32_t r = 0; r < c->ent_count; ++r) {
            const uint16_t ant = p->h_ent_ant[c->ent_begin + r];
            for (uint16_t g : grp_ants) cost += (g == ant) ? -8 : ((g % G) == (ant % G) ? 1 : 0);
          }
          if (!have || cost < best) {
            have = true;
            best = cost;
            pick = i;
          }
        }
      }
      taken[pick] = 1;
      order.push_back(rest[pick]);
      if (const CellRec* c = dense[rest[pick]])
        for (uint32_t r = 0; r < c->ent_count; ++r) grp_ants.push_back(p->h_ent_ant[c->ent_begin + r]);
    }
  }
  p->h_slot_order.insert(p->h_slot_order.end(), order.begin(), order.end());
  // (2) entry order inside each cell
  for (size_t g = 0; g < order.size(); g += G) {
    uint32_t steps = 0;
    for (size_t lane = g; lane < std::min(order.size(), g + G); ++lane) steps = std::max(steps, count_of(order[lane]));
    if (steps == 0) break;
    for (uint32_t step = 0; step < steps; ++step) {
      std::vector<uint16_t> in_bank[G];
      for (size_t lane = g; lane < std::min(order.size(), g + G); ++lane) {
        const CellRec* c = dense[order[lane]];
        if (!c || step >= c->ent_count) continue;
        uint32_t best = step;
        size_t best_cost = ~(size_t)0;
        for (uint32_t r = step; r < c->ent_count; ++r) {
          const uint16_t ant = p->h_ent_ant[c->ent_begin + r];
          const std::vector<uint16_t>& b = in_bank[ant % G];
          const size_t cost = std::find(b.begin(), b.end(), ant) != b.end() ? 0 : b.size();
          if (cost < best_cost) {
            best_cost = cost;
            best = r;
          }
        }
        std::swap(p->h_ent_ant[c->ent_begin + step], p->h_ent_ant[c->ent_begin + best]);
        std::swap(p->h_ent_tap[c->ent_begin + step], p->h_ent_tap[c->ent_begin + best]);
        const uint16_t ant = p->h_ent_ant[c->ent_begin + step];
        std::vector<uint16_t>& b = in_bank[ant % G];
        if (std::find(b.begin(), b.end(), ant) == b.end()) b.push_back(ant);
      }
    }
  }
}

static int build_tables(epic_plan* p, const float* ant_uv_all, const float* taps_all) {
  const int N = p->N, K = p->K, A = p->n_ant, h = (K - 1) / 2, L = p->n_layout;
  const size_t per_layout = (size_t)A * K * K;
  p->cells_host.resize((size_t)L * per_layout);
  // S2 for every layout; the support box is the union of the occupied rows / columns
  std::vector<char> occ_y(N, 0), occ_x(N, 0);
  for (int l = 0; l < L; ++l) {
    const float* ant_uv = ant_uv_all + (size_t)l * A * 2;
    for (int a = 0; a < A; ++a) {
      // reading Q4: nearest cell = floor(double(u) + 0.5)
      const long long cx = (long long)std::floor((double)ant_uv[2 * a + 0] + 0.5);
      const long long cy = (long long)std::floor((double)ant_uv[2 * a + 1] + 0.5);
      for (int iy = 0; iy < K; ++iy)
        for (int ix = 0; ix < K; ++ix) {
          const int y = pos_mod(cy + (iy - h), N); // reading Q6: wrap modulo N
          const int x = pos_mod(cx + (ix - h), N);
          p->cells_host[l * per_layout + ((size_t)a * K + iy) * K + ix] = y * N + x;
          occ_y[y] = 1;
          occ_x[x] = 1;
        }
    }
  }
  circular_box(occ_y, N, &p->y0, &p->R);
  circular_box(occ_x, N, &p->x0, &p->Cc);

  p->h_cells.clear();
  p->h_slot_order.clear();
  p->h_cell_off.assign(1, 0u);
  p->h_ent_ant.resize((size_t)L * per_layout);
  p->h_ent_tap.resize((size_t)L * per_layout);
  std::vector<uint32_t> row_ptr((size_t)L * (p->R + 1), 0);
  std::vector<Entry> ent(per_layout);
  for (int l = 0; l < L; ++l) {
    const float* taps = taps_all ? taps_all + l * per_layout * 2 : nullptr;
    for (int a = 0; a < A; ++a)
      for (int k = 0; k < K * K; ++k) {
        const int cell = p->cells_host[l * per_layout + (size_t)a * K * K + k];
        Entry e;
        e.y = pos_mod(cell / N - p->y0, N);
        e.x = pos_mod(cell % N - p->x0, N);
        e.ant = a;
        e.tap = k;
        ent[(size_t)a * K * K + k] = e;
      }
    std::sort(ent.begin(), ent.end(), [](const Entry& l_, const Entry& r_) {
      if (l_.y != r_.y) return l_.y < r_.y;
      if (l_.x != r_.x) return l_.x < r_.x;
      if (l_.ant != r_.ant) return l_.ant < r_.ant;
      return l_.tap < r_.tap;
    });
    const size_t cell0 = p->h_cells.size(), ent0 = l * per_layout;
    uint32_t* rp = &row_ptr[(size_t)l * (p->R + 1)];
    for (size_t i = 0; i < ent.size(); ++i) {
      const Entry& e = ent[i];
      if (p->h_cells.size() == cell0 || p->h_cells.back().y != e.y || p->h_cells.back().x != e.x) {
        CellRec c;
        c.y = (uint16_t)e.y;
        c.x = (uint16_t)e.x;
        c.ent_begin = (uint32_t)(ent0 + i);
        c.ent_count = 0;
        p->h_cells.push_back(c);
        rp[e.y + 1] += 1;
      }
      p->h_cells.back().ent_count += 1;
      p->h_ent_ant[ent0 + i] = (uint16_t)e.ant;
      float2 w;
      if (taps) {
        w.x = taps[((size_t)e.ant * K * K + e.tap) * 2 + 0];
        w.y = taps[((size_t)e.ant * K * K + e.tap) * 2 + 1];
      } else {
        w.x = 1.0f;
        w.y = 0.0f;
      }
      p->h_ent_tap[ent0 + i] = w;
    }
    if (taps && p->R <= 32 && p->Cc <= 32) bank_order_entries(p, cell0);
    rp[0] = (uint32_t)cell0;  // indices into the concatenated cells array
    for (int y = 0; y < p->R; ++y) rp[y + 1] += rp[y];
    p->h_cell_off.push_back((uint32_t)p->h_cells.size());
  }

  std::vector<float2> tw(N / 2);
  for (int k = 0; k < N / 2; ++k) {
    const double ang = 2.0 * M_PI * (double)k / (double)N; // reading Q8: + sign
    tw[k].x = (float)std::cos(ang);
    tw[k].y = (float)std::sin(ang);
  }

  // one device blob: [cells][row_ptr][ent_tap][twiddle][ent_ant], each 16-byte aligned
  auto align16 = [](size_t v) { return (v + 15) & ~(size_t)15; };
  const size_t o_cells = 0;
  const size_t o_row = align16(o_cells + p->h_cells.size() * sizeof(CellRec));
  const size_t o_tap = align16(o_row + row_ptr.size() * sizeof(uint32_t));
  const size_t o_tw = align16(o_tap + p->h_ent_tap.size() * sizeof(float2));
  const size_t o_ant = align16(o_tw + tw.size() * sizeof(float2));
  const size_t total = align16(o_ant + p->h_ent_ant.size() * sizeof(uint16_t));
  std::vector<char> blob(total, 0);
  std::memcpy(&blob[o_cells], p->h_cells.data(), p->h_cells.size() * sizeof(CellRec));
  std::memcpy(&blob[o_row], row_ptr.data(), row_ptr.size() * sizeof(uint32_t));
  std::memcpy(&blob[o_tap], p->h_ent_tap.data(), p->h_ent_tap.size() * sizeof(float2));
  std::memcpy(&blob[o_tw], tw.data(), tw.size() * sizeof(float2));
  std::memcpy(&blob[o_ant], p->h_ent_ant.data(), p->h_ent_ant.size() * sizeof(uint16_t));
  EPIC_CUDA_TRY(cudaMalloc(&p->d_blob, total));
  EPIC_CUDA_TRY(cudaMemcpy(p->d_blob, blob.data(), total, cudaMemcpyHostToDevice));
  char* d = (char*)p->d_blob;
  DevTables& t = p->t;
  t.cells = (const CellRec*)(d + o_cells);
  t.row_ptr = (const uint32_t*)(d + o_row);
  t.ent_tap = (const float2*)(d + o_tap);
  t.twiddle = (const float2*)(d + o_tw);
  t.ent_ant = (const uint16_t*)(d + o_ant);
  t.n_cells = (int)p->h_cells.size();
  t.n_ent = (int)p->h_ent_ant.size();
  t.N = N;
  t.logN = p->logN;
  t.R = p->R;
  t.Cc = p->Cc;
  t.y0 = p->y0;
  t.x0 = p->x0;
  t.n_ant = A;
  t.is_delta = taps_all ? 0 : 1;
  t.n_layout = L;
  t.row_stride = L > 1 ? p->R + 1 : 0;
  return EPIC_OK;
}

static int resolve_products(const epic_plan* p, int n_pol) {
  if (p->n_products_req == 0) return n_pol == 2 ? 4 : 1;
  return p->n_products_req;
}

static int planes_for(int n_pol, int n_products) {
  if (n_pol == 1 && n_products == 1) return 1;
  if (n_pol == 2 && n_products == 2) return 2;
  if (n_pol == 2 && n_products == 4) return 6;
  return -1;
}

static int image_common(epic_plan* plan, const void* volt, int is_cf32, int n_t, int n_chan,
                        int n_pol, float* out, epic_stream stream) {
  if (!plan) return EPIC_ERR_ARG;
  if (n_t < 0 || n_chan < 0) return EPIC_ERR_ARG;
  if (n_pol != 1 && n_pol != 2) return EPIC_ERR_RANGE;
  const int n_products = resolve_products(plan, n_pol);
  const int n_planes = planes_for(n_pol, n_products);
  if (n_planes < 0) return EPIC_ERR_RANGE;
  plan->last_launches = 0;
  if (plan->n_layout > 1 && n_chan != plan->n_layout) return EPIC_ERR_ARG;  // channel c uses layout c
  if (n_t == 0 || n_chan == 0) return EPIC_OK;
  if (!volt || !out) return EPIC_ERR_ARG;
  ImageArgs a;
  a.volt = volt;
  a.is_cf32 = is_cf32;
  a.native = plan->input_order == EPIC_ORDER_TCAP ? 1 : 0;
  a.phasor = plan->d_phasor;
  a.phasor_pair = plan->d_phasor_pair;
  if (plan->d_phasor && (plan->ph_n_chan != n_chan || plan->ph_n_pol != n_pol)) return EPIC_ERR_ARG;
  a.n_t = n_t;
  a.n_chan = n_chan;
  a.n_pol = n_pol;
  a.n_products = n_products;
  a.n_planes = n_planes;
  a.out = out;
  a.stream = (cudaStream_t)stream;
  const int tiled_can = tiled_supported(plan, is_cf32, n_pol, n_products) &&
                        (reinterpret_cast<uintptr_t>(volt) & 3u) == 0;
  int path = plan->path_req;
  // (the fused kernels fetch bytes when the voltage rows are not word-aligned: any pointer will do)
  const int fused_can = fused_supported(plan, is_cf32, n_pol, n_products);
  const int stream_can = stream_supported(plan, is_cf32, n_pol, n_products);
  // AUTO keeps the batched tiled kernels for N >= 256: measured faster than the streamed kernel;
  // the streamed kernel fetches voltages as bytes, so it takes the antenna counts the tiled row kernel cannot
  if (path == EPIC_PATH_AUTO)
    path = fused_can ? EPIC_PATH_FUSED : (tiled_can ? EPIC_PATH_TILED : (stream_can ? EPIC_PATH_STREAM : EPIC_PATH_TWOPASS));
  if (path == EPIC_PATH_STREAM) {
    if (!stream_can) return EPIC_ERR_RANGE;
    const int st = stream_image(plan, a);
    if (st != EPIC_ERR_RANGE || plan->path_req == EPIC_PATH_STREAM) return st;
    path = EPIC_PATH_TWOPASS;  // AUTO: co-residency is decided at launch
  }
  if (path == EPIC_PATH_FUSED) {
    if (!fused_can) return EPIC_ERR_RANGE;
    return fused_image(plan, a);
  }
  if (path == EPIC_PATH_TILED) {
    if (!tiled_can) return EPIC_ERR_RANGE;
    return tiled_image(plan, a);
  }
  if (path == EPIC_PATH_TENSOR) {
    if (!fused_can || !tensor_supported(plan, is_cf32, n_pol, n_products)) return EPIC_ERR_RANGE;
    return tensor_image(plan, a);
  }
  return twopass_image(plan, a);
}

static void host_pipe_free(epic_plan* plan) {
  HostPipe* hp = plan->pipe;
  if (!hp) return;
  for (int i = 0; i < 2; ++i) {
    if (hp->d_volt[i]) cudaFree(hp->d_volt[i]);
    if (hp->copied[i]) cudaEventDestroy(hp->copied[i]);
    if (hp->consumed[i]) cudaEventDestroy(hp->consumed[i]);
  }
  if (hp->d_out) cudaFree(hp->d_out);
  if (hp->compute) cudaStreamDestroy(hp->compute);
  if (hp->copy) cudaStreamDestroy(hp->copy);
  if (hp->back) cudaStreamDestroy(hp->back);
  delete hp;
  plan->pipe = nullptr;
}

// streams and events on first use; device buffers grown on demand
static int host_pipe_prepare(epic_plan* plan, size_t chunk_bytes, size_t out_bytes) {
  if (!plan->pipe) {
    HostPipe* hp = new (std::nothrow) HostPipe();
    if (!hp) return EPIC_ERR_NOMEM;
    std::memset(hp, 0, sizeof(*hp));
    plan->pipe = hp;
    EPIC_CUDA_TRY(cudaStreamCreateWithFlags(&hp->compute, cudaStreamNonBlocking));
    EPIC_CUDA_TRY(cudaStreamCreateWithFlags(&hp->copy, cudaStreamNonBlocking));
    EPIC_CUDA_TRY(cudaStreamCreateWithFlags(&hp->back, cudaStreamNonBlocking));
    for (int i = 0; i < 2; ++i) {
      EPIC_CUDA_TRY(cudaEventCreateWithFlags(&hp->copied[i], cudaEventDisableTiming));
      EPIC_CUDA_TRY(cudaEventCreateWithFlags(&hp->consumed[i], cudaEventDisableTiming));
    }
  }
  HostPipe* hp = plan->pipe;
  if (chunk_bytes > hp->volt_bytes) {
    EPIC_CUDA_TRY(cudaDeviceSynchronize());
    for (int i = 0; i < 2; ++i) {
      if (hp->d_volt[i]) cudaFree(hp->d_volt[i]);
      hp->d_volt[i] = nullptr;
    }
    hp->volt_bytes = 0;
    for (int i = 0; i < 2; ++i) {
      const cudaError_t ce = cudaMalloc(&hp->d_volt[i], chunk_bytes);
      if (ce != cudaSuccess) { set_cuda_error(ce); return ce == cudaErrorMemoryAllocation ? EPIC_ERR_NOMEM : EPIC_ERR_CUDA; }
    }
    hp->volt_bytes = chunk_bytes;
  }
  if (out_bytes > hp->out_bytes) {
    EPIC_CUDA_TRY(cudaDeviceSynchronize());
    if (hp->d_out) cudaFree(hp->d_out);
    hp->d_out = nullptr;
    hp->out_bytes = 0;
    const cudaError_t ce = cudaMalloc(&hp->d_out, out_bytes);
    if (ce != cudaSuccess) { set_cuda_error(ce); return ce == cudaErrorMemoryAllocation ? EPIC_ERR_NOMEM : EPIC_ERR_CUDA; }
    hp->out_bytes = out_bytes;
  }
  return EPIC_OK;
}

} // namespace epic

using namespace epic;

extern "C" {

int epic_plan_create(epic_plan** out, int grid_n, int pad, int n_ant, const float* ant_uv,
                     const float* kernel_taps, int kernel_k) {
  return epic_plan_create_per_channel(out, grid_n, pad, n_ant, 1, ant_uv, kernel_taps, kernel_k);
}

int epic_plan_create_per_channel(epic_plan** out, int grid_n, int pad, int n_ant, int n_layout,
                                 const float* ant_uv, const float* kernel_taps, int kernel_k) {
  if (!out) return EPIC_ERR_ARG;
  *out = nullptr;
  if (!ant_uv || grid_n < 1 || pad < 1 || n_layout < 1) return EPIC_ERR_ARG;
  const long long Nll = (long long)grid_n * pad;
  if (Nll < 8 || Nll > 512 || (Nll & (Nll - 1)) != 0) return EPIC_ERR_ARG;
  if (kernel_k < 1 || kernel_k > 15 || (kernel_k % 2) == 0) return EPIC_ERR_ARG;
  if (!kernel_taps && kernel_k != 1) return EPIC_ERR_ARG;
  if (n_ant < 1) return EPIC_ERR_ARG;
  if (n_ant > 65535) return EPIC_ERR_RANGE;
  if ((long long)n_layout * n_ant * kernel_k * kernel_k > (1LL << 30)) return EPIC_ERR_RANGE;
  for (long long i = 0; i < 2LL * n_layout * n_ant; ++i)
    if (!std::isfinite(ant_uv[i]) || std::fabs(ant_uv[i]) > 1.0e9f) return EPIC_ERR_ARG;
  epic_plan* p = new (std::nothrow) epic_plan();
  if (!p) return EPIC_ERR_NOMEM;
  p->grid_n = grid_n;
  p->pad = pad;
  p->N = (int)Nll;
  p->logN = 0;
  while ((1 << p->logN) < p->N) ++p->logN;
  p->n_ant = n_ant;
  p->n_layout = n_layout;
  p->K = kernel_k;
  p->n_products_req = 0;
  p->path_req = EPIC_PATH_AUTO;
  p->last_launches = 0;
  p->d_blob = nullptr;
  p->d_scratch = nullptr;
  p->d_fused = nullptr;
  p->fused_ok = 0;
  p->d_tiled = nullptr;
  p->tiled_ok = 0;
  p->d_wide = nullptr;
  p->wide_ok = 0;
  p->pipe = nullptr;
  p->d_auto = nullptr;
  p->input_order = EPIC_ORDER_TCPA;
  p->ph_n_chan = p->ph_n_pol = 0;
  p->d_phasor = nullptr;
  p->d_phasor_pair = nullptr;
  p->scratch_bytes = 0;
  p->scratch_limit = 0;
  int dev = 0;
  cudaDeviceProp prop;
  cudaError_t ce = cudaGetDevice(&dev);
  if (ce == cudaSuccess) ce = cudaGetDeviceProperties(&prop, dev);
  if (ce != cudaSuccess) {
    set_cuda_error(ce);
    delete p;
    return EPIC_ERR_CUDA;
  }
  p->n_sm = prop.multiProcessorCount;
  int st;
  try {
    st = build_tables(p, ant_uv, kernel_taps);
  } catch (const std::bad_alloc&) {
    st = EPIC_ERR_NOMEM;
  }
  if (st == EPIC_OK) {
    // scratch: the two-pass / tiled intermediate H (at least one dual-pol frame) and the fused
    // path's partial sums.  Large planes get 1 GiB: a batch then spans ~150 time samples per channel,
    // which amortises the per-batch read-modify-write of out_accum (measured: C4 +30 % over 96 MiB).
    const size_t frame = (size_t)2 * p->R * p->N * sizeof(float2);
    const size_t want = p->N >= 256 ? ((size_t)1 << 30) : ((size_t)128 << 20);
    p->scratch_bytes = std::max(want, frame);
    ce = cudaMalloc(&p->d_scratch, p->scratch_bytes);
    if (ce != cudaSuccess) {
      set_cuda_error(ce);
      st = (ce == cudaErrorMemoryAllocation) ? EPIC_ERR_NOMEM : EPIC_ERR_CUDA;
    }
  }
  if (st == EPIC_OK) st = fused_plan_init(p);
  if (st == EPIC_OK) st = wide_plan_init(p);
  if (st == EPIC_OK) st = tiled_plan_init(p);
  if (st == EPIC_OK) st = autocorr_plan_init(p, kernel_taps);
  if (st != EPIC_OK) {
    epic_plan_destroy(p);
    return st;
  }
  *out = p;
  return EPIC_OK;
}

int epic_plan_destroy(epic_plan* plan) {
  if (!plan) return EPIC_OK;
  cudaError_t ce = cudaDeviceSynchronize();
  fused_plan_free(plan);
  wide_plan_free(plan);
  tiled_plan_free(plan);
  autocorr_plan_free(plan);
  host_pipe_free(plan);
  if (plan->d_phasor) cudaFree(plan->d_phasor);
  if (plan->d_phasor_pair) cudaFree(plan->d_phasor_pair);
  if (plan->d_scratch) cudaFree(plan->d_scratch);
  if (plan->d_blob) cudaFree(plan->d_blob);
  delete plan;
  if (ce != cudaSuccess) {
    set_cuda_error(ce);
    return EPIC_ERR_CUDA;
  }
  return EPIC_OK;
}

int epic_plan_set_products(epic_plan* plan, int n_products) {
  if (!plan) return EPIC_ERR_ARG;
  if (n_products != 0 && n_products != 1 && n_products != 2 && n_products != 4) return EPIC_ERR_RANGE;
  plan->n_products_req = n_products;
  return EPIC_OK;
}

int epic_plan_set_input_order(epic_plan* plan, int order) {
  if (!plan || (order != EPIC_ORDER_TCPA && order != EPIC_ORDER_TCAP)) return EPIC_ERR_ARG;
  plan->input_order = order;
  return EPIC_OK;
}

int epic_plan_set_delay_phasors(epic_plan* plan, int n_chan, int n_pol, const float* phasors) {
  if (!plan) return EPIC_ERR_ARG;
  // validate first: a rejected call leaves the active table as it was
  if (phasors && (n_chan < 1 || (n_pol != 1 && n_pol != 2))) return EPIC_ERR_ARG;
  float2* d_new = nullptr;
  float4* d_new_pair = nullptr;
  if (phasors) {
    const size_t A = (size_t)plan->n_ant, n = (size_t)n_chan * n_pol * A;
    std::vector<float4> pair((size_t)n_chan * A);
    for (int c = 0; c < n_chan; ++c)
      for (size_t a = 0; a < A; ++a) {
        const float* lo = phasors + (((size_t)c * n_pol + 0) * A + a) * 2;
        const float* hi = phasors + (((size_t)c * n_pol + (n_pol - 1)) * A + a) * 2;
        pair[(size_t)c * A + a] = make_float4(lo[0], hi[0], lo[1], hi[1]);
      }
    cudaError_t ce = cudaMalloc(&d_new, n * sizeof(float2));
    if (ce == cudaSuccess) ce = cudaMalloc(&d_new_pair, (pair.size() + 4) * sizeof(float4));  // + a padded antenna group (fused unpack)
    if (ce == cudaSuccess) ce = cudaMemset(d_new_pair, 0, (pair.size() + 4) * sizeof(float4));
    if (ce == cudaSuccess) ce = cudaMemcpy(d_new, phasors, n * sizeof(float2), cudaMemcpyHostToDevice);
    if (ce == cudaSuccess) ce = cudaMemcpy(d_new_pair, pair.data(), pair.size() * sizeof(float4), cudaMemcpyHostToDevice);
    if (ce != cudaSuccess) {
      set_cuda_error(ce);
      if (d_new) cudaFree(d_new);
      if (d_new_pair) cudaFree(d_new_pair);
      return ce == cudaErrorMemoryAllocation ? EPIC_ERR_NOMEM : EPIC_ERR_CUDA;
    }
  }
  // swap: earlier calls may still read the old table
  const cudaError_t se = cudaDeviceSynchronize();
  if (se != cudaSuccess) {
    set_cuda_error(se);
    if (d_new) cudaFree(d_new);
    if (d_new_pair) cudaFree(d_new_pair);
    return EPIC_ERR_CUDA;
  }
  if (plan->d_phasor) cudaFree(plan->d_phasor);
  if (plan->d_phasor_pair) cudaFree(plan->d_phasor_pair);
  plan->d_phasor = d_new;
  plan->d_phasor_pair = d_new_pair;
  plan->ph_n_chan = phasors ? n_chan : 0;
  plan->ph_n_pol = phasors ? n_pol : 0;
  return EPIC_OK;
}

int epic_plan_set_scratch_limit(epic_plan* plan, long long bytes) {
  if (!plan || bytes < 0) return EPIC_ERR_ARG;
  plan->scratch_limit = (size_t)bytes;
  return EPIC_OK;
}

int epic_plan_set_path(epic_plan* plan, int path) {
  if (!plan) return EPIC_ERR_ARG;
  if (path != EPIC_PATH_AUTO && path != EPIC_PATH_TWOPASS && path != EPIC_PATH_FUSED && path != EPIC_PATH_TILED &&
      path != EPIC_PATH_TENSOR && path != EPIC_PATH_STREAM)
    return EPIC_ERR_ARG;
  if (path == EPIC_PATH_TENSOR && (!plan->fused_ok || plan->N != 128 || plan->n_layout != 1)) return EPIC_ERR_RANGE;
  if (path == EPIC_PATH_FUSED && !plan->fused_ok && !plan->wide_ok) return EPIC_ERR_RANGE;
  if ((path == EPIC_PATH_TILED || path == EPIC_PATH_STREAM) && !plan->tiled_ok) return EPIC_ERR_RANGE;
  plan->path_req = path;
  return EPIC_OK;
}

int epic_image(epic_plan* plan, const void* voltages, int n_t, int n_chan, int n_pol,
               float* out_accum, epic_stream stream) {
  return image_common(plan, voltages, 0, n_t, n_chan, n_pol, out_accum, stream);
}

int epic_image_host(epic_plan* plan, const void* voltages_host, int n_t, int n_chan, int n_pol,
                    float* out_accum_host, int accumulate, int n_chunks) {
  if (!plan) return EPIC_ERR_ARG;
  if (n_t < 0 || n_chan < 0) return EPIC_ERR_ARG;
  if (n_pol != 1 && n_pol != 2) return EPIC_ERR_RANGE;
  const int n_planes = planes_for(n_pol, resolve_products(plan, n_pol));
  if (n_planes < 0) return EPIC_ERR_RANGE;
  plan->last_launches = 0;
  if (plan->n_layout > 1 && n_chan != plan->n_layout) return EPIC_ERR_ARG;
  if (n_chan == 0) return EPIC_OK;
  if (!out_accum_host || (n_t > 0 && !voltages_host)) return EPIC_ERR_ARG;
  const size_t sample_bytes = (size_t)n_chan * n_pol * plan->n_ant;  // one time sample of all channels
  const size_t out_bytes = (size_t)n_chan * n_planes * plan->N * plan->N * sizeof(float);
  // Two ways to cut the gulp.  By CHANNEL range (one-layout plans without delay phasors, enough channels): a chunk's
  // images are final when its kernels end, so the device->host copy of chunk k overlaps the kernels of chunk k+1 just
  // as the host->device copy of chunk k+1 overlaps those of chunk k; the chunk's voltages are a strided slice of the
  // host array ([T][C][Np][A]: one 2-D copy).  By TIME otherwise: the images are read back once, at the end.
  // Automatic chunk count: the first chunk's copy is exposed and every chunk costs a call (launches, fix-up), so
  // n ~ sqrt(bytes / 8 MB), 1..8; sqrt(bytes / 4 MB) for the channel cut, whose read-back overlaps too.
  const bool chan_ok = plan->n_layout == 1 && !plan->d_phasor && n_t > 0;
  if (n_chunks <= 0) {  // measured on C2 (65.5 MB), channel cut: 2 chunks 30.0, 3 31.1, 4 31.5, 6 31.1, 8 30.1 M frames/s
    const double bytes = (double)n_t * (double)sample_bytes;
    n_chunks = std::max(1, std::min(8, (int)std::sqrt(bytes / (chan_ok ? 4.0e6 : 8.0e6))));
  }
  const bool by_channel = chan_ok && n_chan >= 2 * n_chunks && n_chunks > 1;
  const int extent = by_channel ? n_chan : n_t;
  n_chunks = std::max(1, std::min(n_chunks, extent));
  // chunk edges: a short first chunk (its copy is the one nothing can hide), the rest equal
  std::vector<int> edge(1, 0);
  const int first = (n_chunks > 1 && extent >= 4 * n_chunks) ? extent / (2 * n_chunks) : 0;
  if (first) edge.push_back(first);
  const int rest = n_chunks - (first ? 1 : 0);
  for (int k = 1; k <= rest; ++k) edge.push_back(first + (int)((long long)(extent - first) * k / rest));
  int chunk_max = 0;
  for (size_t k = 0; k + 1 < edge.size(); ++k) chunk_max = std::max(chunk_max, edge[k + 1] - edge[k]);
  const size_t chan_bytes = (size_t)n_pol * plan->n_ant;                       // one channel of one time sample
  const size_t img_floats = (size_t)n_planes * plan->N * plan->N;              // one channel's images
  const size_t chunk_bytes = by_channel ? (size_t)chunk_max * chan_bytes * n_t : (size_t)chunk_max * sample_bytes;
  int st = host_pipe_prepare(plan, std::max<size_t>(16, chunk_bytes), out_bytes);
  if (st != EPIC_OK) return st;
  HostPipe* hp = plan->pipe;
  int launches = 0;
  const uint8_t* src = static_cast<const uint8_t*>(voltages_host);
  if (by_channel) {
    for (size_t k = 0; k + 1 < edge.size(); ++k) {
      const int c0 = edge[k], c1 = edge[k + 1], buf = (int)(k & 1);
      if (c1 == c0) continue;
      const size_t width = (size_t)(c1 - c0) * chan_bytes;
      float* d_img = hp->d_out + (size_t)c0 * img_floats;
      const size_t img_bytes = (size_t)(c1 - c0) * img_floats * sizeof(float);
      if (k >= 2) EPIC_CUDA_TRY(cudaStreamWaitEvent(hp->copy, hp->consumed[buf], 0));  // the kernels that read this buffer are done
      EPIC_CUDA_TRY(cudaMemcpy2DAsync(hp->d_volt[buf], width, src + (size_t)c0 * chan_bytes, sample_bytes, width, (size_t)n_t,
                                      cudaMemcpyHostToDevice, hp->copy));
      if (accumulate)
        EPIC_CUDA_TRY(cudaMemcpyAsync(d_img, out_accum_host + (size_t)c0 * img_floats, img_bytes, cudaMemcpyHostToDevice, hp->copy));
      EPIC_CUDA_TRY(cudaEventRecord(hp->copied[buf], hp->copy));
      if (!accumulate) EPIC_CUDA_TRY(cudaMemsetAsync(d_img, 0, img_bytes, hp->compute));
      EPIC_CUDA_TRY(cudaStreamWaitEvent(hp->compute, hp->copied[buf], 0));
      st = image_common(plan, hp->d_volt[buf], 0, n_t, c1 - c0, n_pol, d_img, hp->compute);
      if (st != EPIC_OK) break;
      launches += plan->last_launches;
      EPIC_CUDA_TRY(cudaEventRecord(hp->consumed[buf], hp->compute));
      EPIC_CUDA_TRY(cudaStreamWaitEvent(hp->back, hp->consumed[buf], 0));  // (waits for the record just made, not for later ones)
      EPIC_CUDA_TRY(cudaMemcpyAsync(out_accum_host + (size_t)c0 * img_floats, d_img, img_bytes, cudaMemcpyDeviceToHost, hp->back));
    }
  } else {
    if (accumulate) EPIC_CUDA_TRY(cudaMemcpyAsync(hp->d_out, out_accum_host, out_bytes, cudaMemcpyHostToDevice, hp->compute));
    else EPIC_CUDA_TRY(cudaMemsetAsync(hp->d_out, 0, out_bytes, hp->compute));
    for (size_t k = 0; k + 1 < edge.size(); ++k) {
      const int a = edge[k], b = edge[k + 1], buf = (int)(k & 1);
      if (b == a) continue;
      if (k >= 2) EPIC_CUDA_TRY(cudaStreamWaitEvent(hp->copy, hp->consumed[buf], 0));  // the kernels that read this buffer are done
      EPIC_CUDA_TRY(cudaMemcpyAsync(hp->d_volt[buf], src + (size_t)a * sample_bytes, (size_t)(b - a) * sample_bytes,
                                    cudaMemcpyHostToDevice, hp->copy));
      EPIC_CUDA_TRY(cudaEventRecord(hp->copied[buf], hp->copy));
      EPIC_CUDA_TRY(cudaStreamWaitEvent(hp->compute, hp->copied[buf], 0));
      st = image_common(plan, hp->d_volt[buf], 0, b - a, n_chan, n_pol, hp->d_out, hp->compute);
      if (st != EPIC_OK) break;
      launches += plan->last_launches;
      EPIC_CUDA_TRY(cudaEventRecord(hp->consumed[buf], hp->compute));
    }
    if (st == EPIC_OK) EPIC_CUDA_TRY(cudaMemcpyAsync(out_accum_host, hp->d_out, out_bytes, cudaMemcpyDeviceToHost, hp->compute));
  }
  const cudaError_t c1e = cudaStreamSynchronize(hp->copy), c2e = cudaStreamSynchronize(hp->compute), c3e = cudaStreamSynchronize(hp->back);
  if (st != EPIC_OK) return st;
  if (c1e != cudaSuccess || c2e != cudaSuccess || c3e != cudaSuccess) {
    set_cuda_error(c1e != cudaSuccess ? c1e : (c2e != cudaSuccess ? c2e : c3e));
    return EPIC_ERR_CUDA;
  }
  plan->last_launches = launches;
  return EPIC_OK;
}

int epic_image_noalloc(epic_plan* plan, const void* voltages, int n_t, int n_chan, int n_pol,
                       float* out_accum, epic_stream stream) {
  if (!plan) return EPIC_ERR_ARG;
  if (n_t < 0 || n_chan < 0) return EPIC_ERR_ARG;
  if (n_pol != 1 && n_pol != 2) return EPIC_ERR_RANGE;
  const int n_products = resolve_products(plan, n_pol);
  const int n_planes = planes_for(n_pol, n_products);
  if (n_planes < 0) return EPIC_ERR_RANGE;
  plan->last_launches = 0;
  // the residue-group kernel of epic_fused.cu: one layout, occupied cells within 32 x 32, N = 64 or 128
  if (!plan->fused_ok || plan->N < 64 || plan->n_layout != 1 || !fused_supported(plan, 0, n_pol, n_products)) return EPIC_ERR_RANGE;
  if (plan->d_phasor && (plan->ph_n_chan != n_chan || plan->ph_n_pol != n_pol)) return EPIC_ERR_ARG;
  if (n_t > 0 && n_chan > 0) {
    if (!voltages || !out_accum) return EPIC_ERR_ARG;
  }
  ImageArgs a;
  a.volt = voltages;
  a.is_cf32 = 0;
  a.native = plan->input_order == EPIC_ORDER_TCAP ? 1 : 0;
  a.phasor = plan->d_phasor;
  a.phasor_pair = plan->d_phasor_pair;
  a.n_t = n_t;
  a.n_chan = n_chan;
  a.n_pol = n_pol;
  a.n_products = n_products;
  a.n_planes = n_planes;
  a.out = out_accum;
  a.stream = (cudaStream_t)stream;
  return fused_image_noalloc(plan, a);  // looks the scratch address up (once per device), then n_t == 0 is a no-op
}

long long epic_noalloc_scratch_bytes(void) { return noalloc_scratch_bytes(); }

int epic_image_cf32(epic_plan* plan, const void* voltages_cf32, int n_t, int n_chan, int n_pol,
                    float* out_accum, epic_stream stream) {
  return image_common(plan, voltages_cf32, 1, n_t, n_chan, n_pol, out_accum, stream);
}

int epic_autocorr_remove(epic_plan* plan, const void* voltages, int n_t, int n_chan, int n_pol,
                         float* out_accum, epic_stream stream) {
  if (!plan) return EPIC_ERR_ARG;
  if (n_t < 0 || n_chan < 0) return EPIC_ERR_ARG;
  if (n_pol != 1 && n_pol != 2) return EPIC_ERR_RANGE;
  const int n_products = resolve_products(plan, n_pol);
  const int n_planes = planes_for(n_pol, n_products);
  if (n_planes < 0) return EPIC_ERR_RANGE;
  plan->last_launches = 0;
  if (plan->n_layout > 1 && n_chan != plan->n_layout) return EPIC_ERR_ARG;
  if (n_t == 0 || n_chan == 0) return EPIC_OK;
  if (!voltages || !out_accum) return EPIC_ERR_ARG;
  ImageArgs a;
  a.volt = voltages;
  a.is_cf32 = 0;
  a.native = plan->input_order == EPIC_ORDER_TCAP ? 1 : 0;
  a.phasor = plan->d_phasor;
  a.phasor_pair = plan->d_phasor_pair;
  if (plan->d_phasor && (plan->ph_n_chan != n_chan || plan->ph_n_pol != n_pol)) return EPIC_ERR_ARG;
  a.n_t = n_t;
  a.n_chan = n_chan;
  a.n_pol = n_pol;
  a.n_products = n_products;
  a.n_planes = n_planes;
  a.out = out_accum;
  a.stream = (cudaStream_t)stream;
  return autocorr_remove(plan, a);
}

int epic_plan_get_n(const epic_plan* plan) { return plan ? plan->N : (int)EPIC_ERR_ARG; }

int epic_plan_get_n_layouts(const epic_plan* plan) { return plan ? plan->n_layout : (int)EPIC_ERR_ARG; }

int epic_plan_get_n_planes(const epic_plan* plan, int n_pol) {
  if (!plan) return EPIC_ERR_ARG;
  if (n_pol != 1 && n_pol != 2) return EPIC_ERR_RANGE;
  const int pl = planes_for(n_pol, resolve_products(plan, n_pol));
  return pl < 0 ? (int)EPIC_ERR_RANGE : pl;
}

int epic_plan_get_cells(const epic_plan* plan, int* cells_host) {
  if (!plan || !cells_host) return EPIC_ERR_ARG;
  std::memcpy(cells_host, plan->cells_host.data(), plan->cells_host.size() * sizeof(int));
  return EPIC_OK;
}

int epic_plan_get_support(const epic_plan* plan, int* box_host) {
  if (!plan || !box_host) return EPIC_ERR_ARG;
  box_host[0] = plan->y0;
  box_host[1] = plan->x0;
  box_host[2] = plan->R;
  box_host[3] = plan->Cc;
  return EPIC_OK;
}

int epic_plan_get_path(const epic_plan* plan, int n_pol) {
  if (!plan) return EPIC_ERR_ARG;
  if (n_pol != 1 && n_pol != 2) return EPIC_ERR_RANGE;
  const int n_products = resolve_products(plan, n_pol);
  if (planes_for(n_pol, n_products) < 0) return EPIC_ERR_RANGE;
  if (plan->path_req != EPIC_PATH_AUTO) return plan->path_req;
  if (fused_supported(plan, 0, n_pol, n_products)) return EPIC_PATH_FUSED;
  if (tiled_supported(plan, 0, n_pol, n_products)) return EPIC_PATH_TILED;
  return stream_supported(plan, 0, n_pol, n_products) ? EPIC_PATH_STREAM : EPIC_PATH_TWOPASS;
}

int epic_plan_last_launches(const epic_plan* plan) { return plan ? plan->last_launches : (int)EPIC_ERR_ARG; }

int epic_debug_unpack(const void* bytes_dev, long n, float* out_dev, epic_stream stream) {
  if (n < 0) return EPIC_ERR_ARG;
  if (n == 0) return EPIC_OK;
  if (!bytes_dev || !out_dev) return EPIC_ERR_ARG;
  return debug_unpack(bytes_dev, n, out_dev, (cudaStream_t)stream);
}

int epic_debug_grid_layout(epic_plan* plan, int layout, const void* voltages, int is_cf32, int n_pol,
                           float* out_plane_dev, epic_stream stream) {
  if (!plan || !voltages || !out_plane_dev) return EPIC_ERR_ARG;
  if (layout < 0 || layout >= plan->n_layout) return EPIC_ERR_ARG;
  if (n_pol != 1 && n_pol != 2) return EPIC_ERR_RANGE;
  return debug_grid(plan, layout, voltages, is_cf32 ? 1 : 0, n_pol, out_plane_dev, (cudaStream_t)stream);
}

int epic_debug_grid(epic_plan* plan, const void* voltages, int is_cf32, int n_pol,
                    float* out_plane_dev, epic_stream stream) {
  return epic_debug_grid_layout(plan, 0, voltages, is_cf32, n_pol, out_plane_dev, stream);
}

int epic_fp32_peak_probe(int iters, float* ms_out, double* flops_out) {
  if (iters < 1 || !ms_out || !flops_out) return EPIC_ERR_ARG;
  return fp32_probe(iters, ms_out, flops_out);
}

const char* epic_status_string(int status) {
  switch (status) {
    case EPIC_OK: return "EPIC_OK";
    case EPIC_ERR_ARG: return "EPIC_ERR_ARG: null pointer or invalid shape argument";
    case EPIC_ERR_RANGE: return "EPIC_ERR_RANGE: value outside the supported range";
    case EPIC_ERR_CUDA: return "EPIC_ERR_CUDA: a CUDA runtime call failed";
    case EPIC_ERR_NOMEM: return "EPIC_ERR_NOMEM: allocation failed";
    case EPIC_ERR_SCRATCH: return "EPIC_ERR_SCRATCH: the call needs more than the static scratch of epic_image_noalloc (epic_noalloc_scratch_bytes()) holds";
    default: return "unknown epic_status";
  }
}

int epic_last_cuda_error(void) { return g_last_cuda_error; }

} // extern "C"
