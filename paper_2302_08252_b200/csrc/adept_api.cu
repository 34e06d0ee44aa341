// C ABI of the library (include/adept.h): host-side driver of the transport iterations.
//
// SURVEY.md §8(a) rows A0/A11 on the host side: the host only enqueues step kernels; the counts
// that decide how much work an iteration has live in the device control block, so an iteration
// needs no host round trip.  adept_run reads the control block back every few iterations to test
// for termination (the loop ends when no track is left in any buffer).
#include <algorithm>
#include <cmath>
#include <cstdio>
#include <cstring>
#include <new>
#include <string>
#include <vector>

#include <cuda.h>
#include <cudaTypedefs.h>
#include <cuda_runtime.h>

#include "../../include/adept.h"
#include "step_impl.cuh"

namespace adept {

static thread_local std::string g_create_error;

constexpr size_t kAlign = 256;
constexpr uint32_t kStageRecords = 1u << 20;  // staging chunk for inject / load / read
constexpr size_t kStageRecordBytes = 56;      // max(sizeof(PackedTrack), sizeof(StagedPrimary))
static_assert(sizeof(PackedTrack) == 56 && sizeof(StagedPrimary) == 40, "staged record sizes");
static_assert(sizeof(adept_track) == sizeof(PackedTrack) && sizeof(adept_primary) == 32, "ABI record sizes");

inline size_t align_up(size_t x) { return (x + kAlign - 1) / kAlign * kAlign; }

struct Plan {  // carve-up of the workspace
  size_t ctl, tables, stage, stage_slots;
  size_t rec[3], queue[3][2], ring[3], msc[3];
  size_t instr_rw, instr_lines[3], instr_slots[3];
  size_t total;
  uint32_t capacity;       // rounded up to a multiple of 128 (one tile)
  uint32_t stage_records;
  size_t table_bytes;
  size_t rec_words;        // words of ONE record buffer
  size_t lines_per_kind, slots_per_kind;
  int nbuf;
};

static const LayoutOps *ops_for(int layout) {
  switch (layout) {
    case ADEPT_AOS: return &kOpsAoS;
    case ADEPT_SOA: return &kOpsSoA;
    case ADEPT_AOSOA32: return &kOpsAoSoA32;
    case ADEPT_SOA16: return &kOpsSoA16;
    case ADEPT_HC16: return &kOpsHC16;
    case ADEPT_AOSOA64: return &kOpsAoSoA64;
    case ADEPT_AOSOA16: return &kOpsAoSoA16;
    case ADEPT_AOSOA128: return &kOpsAoSoA128;
    case ADEPT_AOSOA8: return &kOpsAoSoA8;
    default: return nullptr;
  }
}

static bool make_plan(const adept_geometry *g, const adept_tables *t, const adept_config *c, Plan &pl) {
  if (!g || !t || !c) return false;
  const LayoutOps *ops = ops_for(c->layout);
  if (!ops) return false;
  if (c->scheme != ADEPT_SPARSE_SINGLE && c->scheme != ADEPT_DENSE_DOUBLE) return false;
  if (c->flags & ~uint32_t(ADEPT_FLAG_RECYCLE_SLOTS)) return false;
  if (g->n_layers == 0 || g->n_layers > 2048) return false;
  if (t->n_bins == 0 || t->n_bins > 4096 || t->n_materials == 0 || t->n_materials > 8) return false;
  if (t->physics > 2u || (t->physics >= 1u && (c->instrument || (c->flags & ADEPT_FLAG_RECYCLE_SLOTS)))) return false;
  if (c->capacity_per_kind == 0 || c->capacity_per_kind > (1u << 30)) return false;
  pl.capacity = (c->capacity_per_kind + 127u) / 128u * 128u;
  pl.nbuf = (c->scheme == ADEPT_DENSE_DOUBLE) ? 2 : 1;
  pl.rec_words = ops->record_words(pl.capacity);
  // device tables: group 0 = gamma, 1 = e+-, and under the extended physics 2 = e+ extras (rule X38)
  pl.table_bytes = size_t(t->n_materials) * (t->physics ? 3 : 2) * (t->n_bins + 1) * sizeof(float4);
  pl.stage_records = std::min<uint32_t>(pl.capacity, kStageRecords);
  size_t off = 0;
  // control header, tallies (per slab + escaped), section clocks of the timing build
  pl.ctl = off; off = align_up(off + kCtlHeaderBytes + (size_t(2) * g->n_layers + 1 + kNumSections + 4) * sizeof(unsigned long long));
  pl.tables = off; off = align_up(off + pl.table_bytes);
  pl.stage = off; off = align_up(off + size_t(pl.stage_records) * kStageRecordBytes);
  pl.stage_slots = off; off = align_up(off + size_t(pl.stage_records) * 4);
  for (int k = 0; k < 3; ++k) {
    pl.rec[k] = off; off = align_up(off + pl.rec_words * 4 * pl.nbuf);
    for (int q = 0; q < 2; ++q) {
      pl.queue[k][q] = off;
      if (c->scheme == ADEPT_SPARSE_SINGLE) off = align_up(off + size_t(pl.capacity) * 4);
    }
    pl.msc[k] = off;    // rule X39: the three multiple-scattering words of e- / e+ tracks, [buffer][3][capacity]
    if (t->physics == 2u && k != K_GAMMA) off = align_up(off + size_t(pl.capacity) * 3 * sizeof(float) * pl.nbuf);
    pl.ring[k] = off;   // freed slots (ADEPT_FLAG_RECYCLE_SLOTS)
    if (c->scheme == ADEPT_SPARSE_SINGLE && (c->flags & ADEPT_FLAG_RECYCLE_SLOTS)) off = align_up(off + size_t(pl.capacity) * 4);
  }
  pl.lines_per_kind = (pl.rec_words * 4 * pl.nbuf + 127) / 128;
  pl.slots_per_kind = size_t(pl.capacity) * pl.nbuf;
  pl.instr_rw = off;
  if (c->instrument) {
    off = align_up(off + 3 * kNumFields * 2 * sizeof(unsigned long long));
    for (int k = 0; k < 3; ++k) { pl.instr_lines[k] = off; off = align_up(off + pl.lines_per_kind * 4); }
    for (int k = 0; k < 3; ++k) { pl.instr_slots[k] = off; off = align_up(off + pl.slots_per_kind * 4); }
  } else {
    for (int k = 0; k < 3; ++k) pl.instr_lines[k] = pl.instr_slots[k] = off;
  }
  pl.total = off;
  return true;
}

}  // namespace adept

using namespace adept;

struct adept_ctx {
  adept_geometry geo;
  adept_tables tab;       // data pointer not kept
  adept_config cfg;
  Plan plan;
  const LayoutOps *ops;
  Params params;
  cudaStream_t stream;
  // host <-> device record transfers alternate between the two halves of the staging block: the copy
  // of one half (on copy_stream) overlaps the pack/unpack kernel of the other (on `stream`)
  cudaStream_t copy_stream;
  cudaEvent_t ev_copied[2], ev_kernel[2];
  struct Shape { int threads; unsigned grid; size_t dyn_smem; } small, large;  // CTA shapes of the step kernel
  uint64_t live_hint;     // live tracks as last seen by the host: picks the shape
  uint32_t launch_index;  // index of the next step launch (Params::it): the device's iteration counters are kept by it
  unsigned char *ws;
  unsigned char *pinned;  // kCtlHeaderBytes + tallies
  size_t pinned_bytes;
  std::vector<adept_primary> pending;
  size_t pending_done;
  unsigned long long next_primary;
  double e_injected;
  float pitch, depth;
  bool dead;              // after a capacity overflow
  std::string err;
};

namespace {

void free_host_side(adept_ctx *c) {
  if (c->pinned) cudaFreeHost(c->pinned);
  if (c->copy_stream) cudaStreamDestroy(c->copy_stream);
  for (int h = 0; h < 2; ++h) {
    if (c->ev_copied[h]) cudaEventDestroy(c->ev_copied[h]);
    if (c->ev_kernel[h]) cudaEventDestroy(c->ev_kernel[h]);
  }
  delete c;
}

int fail(adept_ctx *c, int code, const char *what, cudaError_t e = cudaSuccess) {
  if (c) {
    c->err = what;
    if (e != cudaSuccess) { c->err += ": "; c->err += cudaGetErrorString(e); }
  }
  return code;
}
#define CU(c, call)                                                   \
  do {                                                                \
    cudaError_t e_ = (call);                                          \
    if (e_ != cudaSuccess) return fail((c), ADEPT_ECUDA, #call, e_);  \
  } while (0)

Ctl *host_ctl(adept_ctx *c) { return reinterpret_cast<Ctl *>(c->pinned); }

__global__ void close_kernel(Params p, uint32_t it, int sparse, int recycle);

// close the open launches (close_kernel), copy control block (+ edep) to pinned memory and wait
int fetch_ctl(adept_ctx *c, bool with_edep) {
  const size_t n = with_edep ? c->pinned_bytes : kCtlHeaderBytes;
  close_kernel<<<1, 32, 0, c->stream>>>(c->params, c->launch_index, c->cfg.scheme == ADEPT_SPARSE_SINGLE ? 1 : 0, int(c->params.recycle));
  CU(c, cudaGetLastError());
  CU(c, cudaMemcpyAsync(c->pinned, c->ws + c->plan.ctl, n, cudaMemcpyDeviceToHost, c->stream));
  CU(c, cudaStreamSynchronize(c->stream));
  c->live_hint = uint64_t(host_ctl(c)->n_cur[0]) + host_ctl(c)->n_cur[1] + host_ctl(c)->n_cur[2];
  if (host_ctl(c)->overflow) {
    c->dead = true;
    return fail(c, ADEPT_ECAPACITY, "track buffer capacity exceeded");
  }
  return ADEPT_OK;
}

void fill_counts(const adept_ctx *c, adept_counts *out) {
  const Ctl *h = reinterpret_cast<const Ctl *>(c->pinned);
  for (int k = 0; k < 3; ++k) {
    out->live[k] = h->n_cur[k];
    out->steps[k] = h->steps[k];
    out->secondaries[k] = h->secondaries[k];
    out->killed[k] = h->killed[k];
    out->escaped_n[k] = h->escaped_n[k];
    out->slots_used[k] = h->slots_used[k];
  }
  out->iterations = h->iterations;
  out->overflow = h->overflow;
  out->reserved = 0;
}

void fill_result(const adept_ctx *c, adept_result *out) {
  const Ctl *h = reinterpret_cast<const Ctl *>(c->pinned);
  fill_counts(c, &out->total);
  out->e_injected = c->e_injected;
  // tallies are 64-bit fixed point on the device (device_state.cuh): per slab, then the escaped energy
  const unsigned long long *fx = reinterpret_cast<const unsigned long long *>(c->pinned + kCtlHeaderBytes);
  const uint32_t n_slabs = 2 * c->geo.n_layers;
  out->e_escaped = double(fx[n_slabs]) * kTallyUnit;
  if (out->edep_slab)
    for (uint32_t s = 0; s < n_slabs; ++s) out->edep_slab[s] = double(fx[s]) * kTallyUnit;
  if (out->edep_layer)
    for (uint32_t l = 0; l < c->geo.n_layers; ++l)
      out->edep_layer[l] = double(fx[2 * l]) * kTallyUnit + double(fx[2 * l + 1]) * kTallyUnit;
}

// write n_cur / slot_top / slots_used of one kind after a host-driven append
__global__ void clear_bad_input_kernel(Ctl *ctl) { ctl->bad_input = 0u; }

// Before the host reads the control block: close every launch that is still open and write the summary.
__global__ void close_kernel(Params p, uint32_t it, int sparse, int recycle) {
  const int lane = int(threadIdx.x);
#ifdef ADEPT_TIMING_SECTIONS
#define ADEPT_ROLL_ARGS p.ctl, p.capacity, it, false, lane, p.sections
#else
#define ADEPT_ROLL_ARGS p.ctl, p.capacity, it, false, lane
#endif
  if (!sparse) roll_iterations<false, false>(ADEPT_ROLL_ARGS);
  else if (recycle) roll_iterations<true, true>(ADEPT_ROLL_ARGS);
  else roll_iterations<true, false>(ADEPT_ROLL_ARGS);
#undef ADEPT_ROLL_ARGS
}

// after a host-driven append: live count of `kind` for the next launch `it`, slot allocator, high-water mark
__global__ void set_counts_kernel(Ctl *ctl, uint32_t it, int kind, uint32_t n_cur, uint32_t slot_top, unsigned long long used) {
  ctl->n[it % 3u][kind] = n_cur;
  ctl->n_cur[kind] = n_cur;
  ctl->slot_top[kind] = slot_top;
  if (used > ctl->slots_used[kind]) ctl->slots_used[kind] = used;
}

__global__ void dev_math_kernel(int fn, const void *in, void *out, unsigned long long n) {
  const unsigned long long i = blockIdx.x * static_cast<unsigned long long>(blockDim.x) + threadIdx.x;
  if (i >= n) return;
  switch (fn) {
    case 0: {
      const uint32_t *a = static_cast<const uint32_t *>(in) + 6 * i;
      static_cast<uint4 *>(out)[i] = philox4x32_10(a[0], a[1], a[2], a[3], a[4], a[5]);
      break;
    }
    case 1: static_cast<float *>(out)[i] = u01(static_cast<const uint32_t *>(in)[i]); break;
    case 2: static_cast<float *>(out)[i] = lg(static_cast<const float *>(in)[i]); break;
    case 3: static_cast<float *>(out)[i] = ex(static_cast<const float *>(in)[i]); break;
    case 4: {
      float s, c;
      sincos2pi(static_cast<const float *>(in)[i], s, c);
      static_cast<float2 *>(out)[i] = make_float2(s, c);
      break;
    }
    default: {
      const float2 ab = static_cast<const float2 *>(in)[i];
      static_cast<float *>(out)[i] = div_rn_inrange(ab.x, ab.y);
    }
  }
}

}  // namespace

// =================================================================== extern "C" =============
extern "C" {

size_t adept_workspace_bytes(const adept_geometry *g, const adept_tables *t, const adept_config *c) {
  Plan pl;
  return make_plan(g, t, c, pl) ? pl.total : 0;
}

const char *adept_last_error(const adept_ctx *c) { return c ? c->err.c_str() : g_create_error.c_str(); }

static int clear_state(adept_ctx *c) {
  // everything except the tables: control block, tallies, instrumentation counters
  const Plan &pl = c->plan;
  CU(c, cudaMemsetAsync(c->ws + pl.ctl, 0, pl.tables - pl.ctl, c->stream));
  if (c->cfg.instrument && pl.total > pl.instr_rw)
    CU(c, cudaMemsetAsync(c->ws + pl.instr_rw, 0, pl.total - pl.instr_rw, c->stream));
#ifdef ADEPT_TIMING_SECTIONS
  {  // scratch of the launch timeline, by launch parity: {earliest CTA start (atomicMin), latest CTA end (atomicMax)}
    static const unsigned long long kInit[4] = {~0ull, 0ull, ~0ull, 0ull};
    CU(c, cudaMemcpyAsync(c->params.sections + kNumSections, kInit, sizeof kInit, cudaMemcpyHostToDevice, c->stream));
  }
#endif
  c->pending.clear();
  c->pending_done = 0;
  c->next_primary = 0;
  c->e_injected = 0.0;
  c->live_hint = 0;
  c->launch_index = 0;
  c->dead = false;
  return ADEPT_OK;
}

int adept_create(const adept_geometry *g, const adept_tables *t, const adept_config *cfg, adept_ctx **out) {
  g_create_error.clear();
  auto bad = [&](const char *why) { g_create_error = why; return ADEPT_EINVAL; };
  if (!out) return bad("out is NULL");
  *out = nullptr;
  Plan pl;
  if (!make_plan(g, t, cfg, pl)) return bad("invalid geometry, tables or configuration");
  if (!t->data) return bad("tables.data is NULL");
  if (t->physics >= 1u && !t->data_x) return bad("tables.physics >= 1 needs tables.data_x");
  if (!(g->abs_mm > 0.0f) || !(g->gap_mm > 0.0f) || !(g->half_xy_mm > 0.0f)) return bad("non-positive geometry");
  if (g->mat_abs >= t->n_materials || g->mat_gap >= t->n_materials) return bad("material index out of range");
  if (!(t->e_cut > 0.0f) || !(t->e_max > t->e_min) || !(t->e_min > 0.0f)) return bad("invalid energy grid");
  if (!cfg->workspace || (reinterpret_cast<uintptr_t>(cfg->workspace) % kAlign) != 0) return bad("workspace must be a 256-byte aligned device pointer");
  if (cfg->workspace_bytes < pl.total) return bad("workspace too small (see adept_workspace_bytes)");

  adept_ctx *c = new (std::nothrow) adept_ctx();
  if (!c) return bad("out of host memory");
  c->geo = *g; c->tab = *t; c->tab.data = nullptr; c->tab.data_x = nullptr; c->cfg = *cfg; c->plan = pl;
  c->ops = ops_for(cfg->layout);
  c->stream = static_cast<cudaStream_t>(cfg->cuda_stream);
  c->ws = static_cast<unsigned char *>(cfg->workspace);
  c->pinned = nullptr;
  c->copy_stream = nullptr;
  for (int h = 0; h < 2; ++h) c->ev_copied[h] = c->ev_kernel[h] = nullptr;
  c->pitch = g->abs_mm + g->gap_mm;
  c->depth = static_cast<float>(g->n_layers) * c->pitch;
  auto die = [&](const char *what, cudaError_t e) {
    g_create_error = std::string(what) + ": " + cudaGetErrorString(e);
    free_host_side(c);
    return ADEPT_ECUDA;
  };
  cudaError_t e;
  c->pinned_bytes = kCtlHeaderBytes + (size_t(2) * g->n_layers + 1 + kNumSections + 4) * sizeof(unsigned long long);
  if ((e = cudaMallocHost(reinterpret_cast<void **>(&c->pinned), c->pinned_bytes)) != cudaSuccess)
    return die("cudaMallocHost", e);
  if ((e = cudaStreamCreateWithFlags(&c->copy_stream, cudaStreamNonBlocking)) != cudaSuccess)
    return die("cudaStreamCreateWithFlags", e);
  for (int h = 0; h < 2; ++h) {
    if ((e = cudaEventCreateWithFlags(&c->ev_copied[h], cudaEventDisableTiming)) != cudaSuccess ||
        (e = cudaEventCreateWithFlags(&c->ev_kernel[h], cudaEventDisableTiming)) != cudaSuccess)
      return die("cudaEventCreateWithFlags", e);
  }

  // tables: [mat][group][qty][node] (host, ABI) -> [group][mat][node]{q0,q1,q2,0} (device): a CTA
  // stages only the group of the particle kind it is stepping, and one 16-byte shared-memory load
  // fetches all three quantities of a node.
  const uint32_t nodes = t->n_bins + 1;
  std::vector<float> packed(pl.table_bytes / sizeof(float), 0.0f);
  for (uint32_t m = 0; m < t->n_materials; ++m)
    for (uint32_t grp = 0; grp < 2; ++grp)
      for (uint32_t q = 0; q < 3; ++q)
        for (uint32_t j = 0; j < nodes; ++j)
          packed[((size_t(grp) * t->n_materials + m) * nodes + j) * 4 + q] = t->data[((size_t(m) * 2 + grp) * 3 + q) * nodes + j];
  if (t->physics >= 1u)  // X36: Sigma_delta in the fourth lane of the e+- group
    for (uint32_t m = 0; m < t->n_materials; ++m)
      for (uint32_t j = 0; j < nodes; ++j)
      {  // data_x[mat][3][node]: Sigma_delta -> fourth lane of the e+- group; Sigma_annihilation, Sigma_transport ->
         // first and second lane of group 2
        packed[((size_t(1) * t->n_materials + m) * nodes + j) * 4 + 3] = t->data_x[(size_t(m) * 3 + 0) * nodes + j];
        packed[((size_t(2) * t->n_materials + m) * nodes + j) * 4 + 0] = t->data_x[(size_t(m) * 3 + 1) * nodes + j];
        packed[((size_t(2) * t->n_materials + m) * nodes + j) * 4 + 1] = t->data_x[(size_t(m) * 3 + 2) * nodes + j];
      }
  if ((e = cudaMemcpyAsync(c->ws + pl.tables, packed.data(), pl.table_bytes, cudaMemcpyHostToDevice, c->stream)) != cudaSuccess)
    return die("cudaMemcpyAsync(tables)", e);
  if ((e = cudaStreamSynchronize(c->stream)) != cudaSuccess) return die("cudaStreamSynchronize", e);

  Params &p = c->params;
  p.ctl = reinterpret_cast<Ctl *>(c->ws + pl.ctl);
  p.tally = reinterpret_cast<unsigned long long *>(c->ws + pl.ctl + kCtlHeaderBytes);
  p.sections = p.tally + (size_t(2) * g->n_layers + 1);
  p.tables = reinterpret_cast<const float4 *>(c->ws + pl.tables);
  p.table_bytes = static_cast<uint32_t>(size_t(t->n_materials) * nodes * sizeof(float4));  // per particle group
  p.table_area = p.table_bytes * (t->physics ? 2u : 1u);
  p.nodes = nodes;
  p.ln_e_min = t->ln_e_min; p.inv_dln = t->inv_dln; p.e_cut = t->e_cut; p.e_max = t->e_max;
  p.n_slabs = 2 * g->n_layers;
  p.abs_mm = g->abs_mm; p.pitch = c->pitch; p.half_xy = g->half_xy_mm;
  p.mat_abs = g->mat_abs; p.mat_gap = g->mat_gap;
  p.capacity = pl.capacity;
  p.recycle = (cfg->scheme == ADEPT_SPARSE_SINGLE && (cfg->flags & ADEPT_FLAG_RECYCLE_SLOTS)) ? 1u : 0u;
  p.physics = t->physics;
  const int variant = (p.recycle ? V_RECYCLE : 0) | (p.physics ? V_PHYS : 0) | (p.physics == 2u ? V_MSC : 0);
  for (int k = 0; k < 3; ++k) {
    uint32_t *r = reinterpret_cast<uint32_t *>(c->ws + pl.rec[k]);
    p.kind[k].rec[0] = r;
    p.kind[k].rec[1] = (pl.nbuf == 2) ? r + pl.rec_words : r;
    p.kind[k].queue[0] = reinterpret_cast<uint32_t *>(c->ws + pl.queue[k][0]);
    p.kind[k].queue[1] = reinterpret_cast<uint32_t *>(c->ws + pl.queue[k][1]);
    p.kind[k].free_ring = reinterpret_cast<uint32_t *>(c->ws + pl.ring[k]);
    p.kind[k].msc[0] = reinterpret_cast<float *>(c->ws + pl.msc[k]);
    p.kind[k].msc[1] = (pl.nbuf == 2) ? p.kind[k].msc[0] + size_t(pl.capacity) * 3 : p.kind[k].msc[0];
    p.kind[k].instr_lines = reinterpret_cast<uint32_t *>(c->ws + pl.instr_lines[k]);
    p.kind[k].instr_slots = reinterpret_cast<uint32_t *>(c->ws + pl.instr_slots[k]);
  }
  p.instr_field_rw = reinterpret_cast<unsigned long long *>(c->ws + pl.instr_rw);
  std::memset(p.tile_map, 0, sizeof p.tile_map);
  if ((cfg->layout == ADEPT_SOA || cfg->layout == ADEPT_AOS) && cfg->scheme == ADEPT_DENSE_DOUBLE) {
    // Tensor maps of the six record buffers: one tiled TMA copy stages a tile (csrc/step_impl.cuh
    // prefetch_tile).  SoA: a [14 fields][capacity] u32 tensor with a box of [14][kGroup].  AoS: a
    // [capacity][16 words] tensor with a box of [kGroup][16], copied with the 64-byte swizzle.
    // The encoder is a driver entry point; it is fetched through the runtime so that the library
    // does not link libcuda.
    void *fn = nullptr;
    cudaDriverEntryPointQueryResult qres;
    if ((e = cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &fn, cudaEnableDefault, &qres)) != cudaSuccess || !fn)
      return die("cudaGetDriverEntryPoint(cuTensorMapEncodeTiled)", e == cudaSuccess ? cudaErrorUnknown : e);
    auto encode = reinterpret_cast<PFN_cuTensorMapEncodeTiled_v12000>(fn);
    const bool soa = cfg->layout == ADEPT_SOA;
    const cuuint64_t dims[2] = {soa ? cuuint64_t(pl.capacity) : 16u, soa ? cuuint64_t(kNumFields) : cuuint64_t(pl.capacity)};
    const cuuint64_t strides[1] = {soa ? cuuint64_t(pl.capacity) * 4 : 64u};  // bytes between rows
    const cuuint32_t box[2] = {soa ? cuuint32_t(kGroup) : 16u, soa ? cuuint32_t(kNumFields) : cuuint32_t(kGroup)};
    const cuuint32_t elem_strides[2] = {1, 1};
    for (int k = 0; k < 3; ++k)
      for (int b = 0; b < 2; ++b) {
        const CUresult r = encode(&p.tile_map[k][b], CU_TENSOR_MAP_DATA_TYPE_UINT32, 2, p.kind[k].rec[b], dims, strides,
                                  box, elem_strides, CU_TENSOR_MAP_INTERLEAVE_NONE,
                                  soa ? CU_TENSOR_MAP_SWIZZLE_NONE : CU_TENSOR_MAP_SWIZZLE_64B,
                                  CU_TENSOR_MAP_L2_PROMOTION_L2_128B, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
        if (r != CUDA_SUCCESS) return die("cuTensorMapEncodeTiled", cudaErrorInvalidValue);
      }
  }

  // persistent grids: as many CTAs as fit on the device at once, for both CTA shapes of the step
  // kernel (device_state.cuh); the large shape is optional (huge tables may not leave room for it)
  int dev = 0, sms = 0;
  if ((e = cudaGetDevice(&dev)) != cudaSuccess) return die("cudaGetDevice", e);
  if ((e = cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev)) != cudaSuccess)
    return die("cudaDeviceGetAttribute", e);
  const int instr = cfg->instrument ? 1 : 0;
  const size_t tile_words = c->ops->record_words(kGroup);
  c->small.threads = kBlockSmall;
  c->small.dyn_smem = step_smem_bytes(cfg->scheme, p.table_area, p.n_slabs, tile_words, kBlockSmall, c->ops->sparse_gather, p.physics == 2u);
  const int per_sm = c->ops->step_ctas_per_sm(cfg->scheme, instr, variant, kBlockSmall, c->small.dyn_smem);
  if (per_sm <= 0) {
    g_create_error = "step kernel does not fit on an SM with these tables (shared memory)";
    free_host_side(c);
    return ADEPT_EINVAL;
  }
  c->small.grid = static_cast<unsigned>(sms * per_sm);
  c->large.threads = kBlockLarge;
  c->large.dyn_smem = step_smem_bytes(cfg->scheme, p.table_area, p.n_slabs, tile_words, kBlockLarge, c->ops->sparse_gather, p.physics == 2u);
  const int per_sm_large = c->ops->step_ctas_per_sm(cfg->scheme, instr, variant, kBlockLarge, c->large.dyn_smem);
  cudaGetLastError();  // a failed attribute query of the optional shape is not an error of the context
  c->large.grid = per_sm_large > 0 ? static_cast<unsigned>(sms * per_sm_large) : 0u;
  c->live_hint = 0;

  int rc = clear_state(c);
  if (rc == ADEPT_OK && (e = cudaStreamSynchronize(c->stream)) != cudaSuccess) rc = ADEPT_ECUDA;
  if (rc != ADEPT_OK) {
    g_create_error = c->err.empty() ? "clearing the workspace failed" : c->err;
    free_host_side(c);
    return rc;
  }
  *out = c;
  return ADEPT_OK;
}

int adept_destroy(adept_ctx *c) {
  if (!c) return ADEPT_EINVAL;
  cudaStreamSynchronize(c->stream);
  cudaStreamSynchronize(c->copy_stream);
  free_host_side(c);
  return ADEPT_OK;
}

int adept_set_primary_index(adept_ctx *c, uint64_t next_index) {
  if (!c) return ADEPT_EINVAL;
  if (c->pending_done < c->pending.size())
    return fail(c, ADEPT_ESTATE, "adept_set_primary_index: primaries are still queued for adept_run");
  c->next_primary = next_index;
  return ADEPT_OK;
}

int adept_reset(adept_ctx *c) {
  if (!c) return ADEPT_EINVAL;
  int rc = clear_state(c);
  if (rc != ADEPT_OK) return rc;
  CU(c, cudaStreamSynchronize(c->stream));
  c->err.clear();
  return ADEPT_OK;
}

// ---- appending tracks from the host --------------------------------------------------------
static int check_alive(adept_ctx *c) {
  if (!c) return ADEPT_EINVAL;
  if (c->dead) return fail(c, ADEPT_ESTATE, "context overflowed: only adept_reset / adept_destroy are accepted");
  return ADEPT_OK;
}

static bool primary_ok(const adept_ctx *c, const adept_primary &p) {
  if (p.kind > 2u) return false;
  if (!(p.pos[2] >= 0.0f) || !(p.pos[2] <= c->depth)) return false;
  if (!(std::fabs(p.pos[0]) <= c->geo.half_xy_mm) || !(std::fabs(p.pos[1]) <= c->geo.half_xy_mm)) return false;
  if (!(p.ekin >= c->tab.e_cut) || !(p.ekin <= c->tab.e_max)) return false;
  return true;
}

// Make `n` validated primaries live (rule R4: ids from the running global index).
static int inject_now(adept_ctx *c, const adept_primary *prim, uint64_t n) {
  if (n == 0) return ADEPT_OK;
  int rc = fetch_ctl(c, false);
  if (rc != ADEPT_OK) return rc;
  const Ctl h = *host_ctl(c);
  const bool sparse = c->cfg.scheme == ADEPT_SPARSE_SINGLE;
  uint32_t n_cur[3], top[3];
  uint64_t add[3] = {0, 0, 0};
  for (uint64_t i = 0; i < n; ++i) add[prim[i].kind] += 1;
  for (int k = 0; k < 3; ++k) {
    n_cur[k] = h.n_cur[k]; top[k] = h.slot_top[k];
    if (n_cur[k] + add[k] > c->plan.capacity || (sparse && top[k] + add[k] > c->plan.capacity))
      return fail(c, ADEPT_ECAPACITY, "adept_inject: more primaries than free capacity");
  }
  std::vector<StagedPrimary> stage;
  for (int k = 0; k < 3; ++k) {
    if (!add[k]) continue;
    stage.clear();
    stage.reserve(add[k]);
    for (uint64_t i = 0; i < n; ++i) {
      if (prim[i].kind != uint32_t(k)) continue;
      StagedPrimary s;
      s.kind = prim[i].kind;
      std::memcpy(s.pos, prim[i].pos, sizeof s.pos);
      std::memcpy(s.dir, prim[i].dir, sizeof s.dir);
      s.ekin = prim[i].ekin;
      s.gidx = c->next_primary + i;
      stage.push_back(s);
    }
    for (uint64_t done = 0; done < add[k];) {
      const uint32_t m = uint32_t(std::min<uint64_t>(add[k] - done, c->plan.stage_records));
      CU(c, cudaMemcpyAsync(c->ws + c->plan.stage, stage.data() + done, size_t(m) * sizeof(StagedPrimary),
                            cudaMemcpyHostToDevice, c->stream));
      CU(c, c->ops->launch_inject(c->cfg.scheme, c->params, c->ws + c->plan.stage, m, k, h.parity, n_cur[k], top[k],
                                  c->cfg.seed, c->stream));
      CU(c, cudaStreamSynchronize(c->stream));  // the staging area and `stage` are reused
      n_cur[k] += m;
      if (sparse) top[k] += m;
      done += m;
    }
    set_counts_kernel<<<1, 1, 0, c->stream>>>(c->params.ctl, c->launch_index, k, n_cur[k], top[k], sparse ? top[k] : n_cur[k]);
    CU(c, cudaGetLastError());
  }
  for (uint64_t i = 0; i < n; ++i)
    c->e_injected += double(prim[i].ekin) + (prim[i].kind == 1u ? double(2.0f * kMc2) : 0.0);
  c->next_primary += n;
  c->live_hint += n;
  return ADEPT_OK;
}

int adept_inject(adept_ctx *c, const adept_primary *prim, uint64_t n) {
  int rc = check_alive(c);
  if (rc != ADEPT_OK) return rc;
  if (n && !prim) return fail(c, ADEPT_EINVAL, "adept_inject: primaries is NULL");
  for (uint64_t i = 0; i < n; ++i)
    if (!primary_ok(c, prim[i])) return fail(c, ADEPT_EINVAL, "adept_inject: primary outside the calorimeter or energy grid");
  if (c->cfg.batch_primaries == 0) return inject_now(c, prim, n);
  c->pending.insert(c->pending.end(), prim, prim + n);
  return ADEPT_OK;
}

int adept_load_tracks(adept_ctx *c, uint32_t kind, const adept_track *tracks, uint64_t n, const uint32_t *slots) {
  int rc = check_alive(c);
  if (rc != ADEPT_OK) return rc;
  if (kind > 2u || (n && !tracks)) return fail(c, ADEPT_EINVAL, "adept_load_tracks: bad kind or NULL tracks");
  if (n == 0) return ADEPT_OK;
  rc = fetch_ctl(c, false);
  if (rc != ADEPT_OK) return rc;
  const Ctl h = *host_ctl(c);
  const bool sparse = c->cfg.scheme == ADEPT_SPARSE_SINGLE;
  const uint32_t cap = c->plan.capacity;
  if (h.n_cur[kind] + n > cap) return fail(c, ADEPT_EINVAL, "adept_load_tracks: more tracks than free capacity");
  uint32_t top = h.slot_top[kind];
  if (sparse) {
    if (slots) {
      // "all distinct, free and < capacity": slots are handed out by a bump allocator (rule S30), so
      // the free ones are exactly those at or above its top; distinctness by a bitmap over them
      std::vector<uint64_t> seen((size_t(cap - h.slot_top[kind]) + 63) / 64, 0ull);
      for (uint64_t i = 0; i < n; ++i) {
        if (slots[i] >= cap) return fail(c, ADEPT_EINVAL, "adept_load_tracks: slot out of range");
        if (slots[i] < h.slot_top[kind]) return fail(c, ADEPT_EINVAL, "adept_load_tracks: slot is not free");
        const uint32_t r = slots[i] - h.slot_top[kind];
        if (seen[r >> 6] & (1ull << (r & 63))) return fail(c, ADEPT_EINVAL, "adept_load_tracks: duplicate slot");
        seen[r >> 6] |= 1ull << (r & 63);
        top = std::max(top, slots[i] + 1u);
      }
    } else {
      if (top + n > cap) return fail(c, ADEPT_EINVAL, "adept_load_tracks: more tracks than free slots");
    }
  }
  // Chunks alternate between the two halves of the staging block: the host-to-device copy of one
  // half (copy_stream) overlaps the unpack kernel of the other (the context's stream).  The records
  // themselves are validated by the unpack kernel (Ctl::bad_input).
  const uint32_t half = std::max<uint32_t>(1u, c->plan.stage_records / 2);
  uint32_t n_cur = h.n_cur[kind], next_slot = h.slot_top[kind];
  CU(c, cudaEventRecord(c->ev_kernel[0], c->stream));   // everything enqueued so far precedes the first copies
  CU(c, cudaEventRecord(c->ev_kernel[1], c->stream));
  int hb = 0;
  for (uint64_t done = 0; done < n; hb ^= 1) {
    const uint32_t m = uint32_t(std::min<uint64_t>(n - done, half));
    unsigned char *stage = c->ws + c->plan.stage + size_t(hb) * half * kStageRecordBytes;
    uint32_t *stage_slots = reinterpret_cast<uint32_t *>(c->ws + c->plan.stage_slots) + size_t(hb) * half;
    CU(c, cudaStreamWaitEvent(c->copy_stream, c->ev_kernel[hb], 0));   // the half's previous chunk was consumed
    CU(c, cudaMemcpyAsync(stage, tracks + done, size_t(m) * sizeof(adept_track), cudaMemcpyHostToDevice, c->copy_stream));
    const uint32_t *dslots = nullptr;
    if (sparse && slots) {
      CU(c, cudaMemcpyAsync(stage_slots, slots + done, size_t(m) * 4, cudaMemcpyHostToDevice, c->copy_stream));
      dslots = stage_slots;
    }
    CU(c, cudaEventRecord(c->ev_copied[hb], c->copy_stream));
    CU(c, cudaStreamWaitEvent(c->stream, c->ev_copied[hb], 0));
    CU(c, c->ops->launch_load(c->cfg.scheme, c->params, stage, dslots, m, int(kind), h.parity, n_cur, next_slot, c->stream));
    CU(c, cudaEventRecord(c->ev_kernel[hb], c->stream));
    n_cur += m;
    next_slot += m;
    done += m;
  }
  rc = fetch_ctl(c, false);   // synchronises: the caller's arrays are free again
  if (rc != ADEPT_OK) return rc;
  if (host_ctl(c)->bad_input) {
    clear_bad_input_kernel<<<1, 1, 0, c->stream>>>(c->params.ctl);
    CU(c, cudaGetLastError());
    CU(c, cudaStreamSynchronize(c->stream));
    return fail(c, ADEPT_EINVAL, "adept_load_tracks: a record breaks the preconditions (vol, step, ekin, dir; see adept.h)");
  }
  if (sparse && !slots) top = next_slot;
  c->live_hint += n;
  set_counts_kernel<<<1, 1, 0, c->stream>>>(c->params.ctl, c->launch_index, int(kind), n_cur, top, sparse ? top : n_cur);
  CU(c, cudaGetLastError());
  return ADEPT_OK;
}

int adept_read_tracks(adept_ctx *c, uint32_t kind, adept_track *out, uint64_t cap, uint64_t *n) {
  if (!c || kind > 2u || !n) return c ? fail(c, ADEPT_EINVAL, "adept_read_tracks: bad argument") : ADEPT_EINVAL;
  int rc = fetch_ctl(c, false);
  if (rc != ADEPT_OK && rc != ADEPT_ECAPACITY) return rc;
  const Ctl h = *host_ctl(c);
  *n = h.n_cur[kind];
  if (*n > cap || (*n && !out)) return fail(c, ADEPT_EINVAL, "adept_read_tracks: output array too small");
  // pack kernel of one half of the staging block (the context's stream) overlaps the device-to-host
  // copy of the other (copy_stream)
  const uint32_t half = std::max<uint32_t>(1u, c->plan.stage_records / 2);
  CU(c, cudaEventRecord(c->ev_copied[0], c->copy_stream));
  CU(c, cudaEventRecord(c->ev_copied[1], c->copy_stream));
  int hb = 0;
  for (uint64_t done = 0; done < *n; hb ^= 1) {
    const uint32_t m = uint32_t(std::min<uint64_t>(*n - done, half));
    unsigned char *stage = c->ws + c->plan.stage + size_t(hb) * half * kStageRecordBytes;
    CU(c, cudaStreamWaitEvent(c->stream, c->ev_copied[hb], 0));   // the half's previous chunk has left
    CU(c, c->ops->launch_read(c->cfg.scheme, c->params, stage, uint32_t(done), m, int(kind), h.parity, c->stream));
    CU(c, cudaEventRecord(c->ev_kernel[hb], c->stream));
    CU(c, cudaStreamWaitEvent(c->copy_stream, c->ev_kernel[hb], 0));
    CU(c, cudaMemcpyAsync(out + done, stage, size_t(m) * sizeof(adept_track), cudaMemcpyDeviceToHost, c->copy_stream));
    CU(c, cudaEventRecord(c->ev_copied[hb], c->copy_stream));
    done += m;
  }
  CU(c, cudaStreamSynchronize(c->copy_stream));
  CU(c, cudaStreamSynchronize(c->stream));
  return rc;
}

// ---- iterations -----------------------------------------------------------------------------
#ifndef ADEPT_LARGE_SHAPE_MIN_TRACKS
#define ADEPT_LARGE_SHAPE_MIN_TRACKS (1u << 22)
#endif
static int launch_iteration(adept_ctx *c) {
  const adept_ctx::Shape &sh = (c->large.grid != 0u && c->live_hint >= ADEPT_LARGE_SHAPE_MIN_TRACKS) ? c->large : c->small;
  c->params.it = c->launch_index;
  c->launch_index = next_launch(c->launch_index);
  CU(c, c->ops->launch_step(c->cfg.scheme, c->cfg.instrument ? 1 : 0, c->params, sh.threads, sh.grid, sh.dyn_smem,
                            c->stream));
  return ADEPT_OK;
}

int adept_step(adept_ctx *c, adept_counts *out) {
  int rc = check_alive(c);
  if (rc != ADEPT_OK) return rc;
  rc = launch_iteration(c);
  if (rc != ADEPT_OK || !out) return rc;
  rc = fetch_ctl(c, false);
  fill_counts(c, out);
  return rc;
}

int adept_get_result(adept_ctx *c, adept_result *out) {
  if (!c || !out) return c ? fail(c, ADEPT_EINVAL, "adept_get_result: out is NULL") : ADEPT_EINVAL;
  const int rc = fetch_ctl(c, true);
  if (rc != ADEPT_OK && rc != ADEPT_ECAPACITY) return rc;
  fill_result(c, out);
  return rc;
}

int adept_run(adept_ctx *c, uint64_t max_iterations, adept_result *out) {
  int rc = check_alive(c);
  if (rc != ADEPT_OK) return rc;
  // Iterations are enqueued in bursts; the control block is read back after each burst.  An
  // iteration with nothing alive is a no-op on the device and is not counted (Ctl::iterations), so
  // over-shooting the end of a batch by a few launches is harmless; progress against
  // max_iterations is what the device counted, not what the host enqueued.
  // A burst boundary costs a stream synchronisation and a host round trip (~ 20 us, measured: config 2
  // 1.84 ms with bursts of 16, 1.72 ms with bursts of 64), an over-shot launch ~ 2.5 us: bursts start at
  // 16 launches and double up to 64 while a batch is alive.
#ifndef ADEPT_RUN_BURST
#define ADEPT_RUN_BURST 16
#endif
#ifndef ADEPT_RUN_BURST_MAX
#define ADEPT_RUN_BURST_MAX 64
#endif
  uint64_t next_burst = ADEPT_RUN_BURST;
  uint64_t first_iteration = 0;
  for (bool first = true;; first = false) {
    rc = fetch_ctl(c, false);
    if (rc != ADEPT_OK) break;
    const Ctl *h = host_ctl(c);
    if (first) first_iteration = h->iterations;
    const uint64_t done = h->iterations - first_iteration;
    if (max_iterations && done >= max_iterations) break;
    const uint64_t live = uint64_t(h->n_cur[0]) + h->n_cur[1] + h->n_cur[2];
    if (live == 0) {
      if (c->pending_done >= c->pending.size()) break;
      const uint64_t batch = std::min<uint64_t>(c->cfg.batch_primaries ? c->cfg.batch_primaries : c->pending.size(),
                                                c->pending.size() - c->pending_done);
      rc = inject_now(c, c->pending.data() + c->pending_done, batch);
      if (rc != ADEPT_OK) break;
      c->pending_done += batch;
      if (c->pending_done >= c->pending.size()) { c->pending.clear(); c->pending_done = 0; }
      next_burst = ADEPT_RUN_BURST;
    }
    uint64_t burst = next_burst;
    next_burst = std::min<uint64_t>(2 * next_burst, ADEPT_RUN_BURST_MAX);
    if (max_iterations) burst = std::min<uint64_t>(burst, max_iterations - done);
    for (uint64_t i = 0; i < burst && rc == ADEPT_OK; ++i) rc = launch_iteration(c);
    if (rc != ADEPT_OK) break;
  }
  if (out && (rc == ADEPT_OK || rc == ADEPT_ECAPACITY)) {
    const int rc2 = fetch_ctl(c, true);
    if (rc2 == ADEPT_OK || rc2 == ADEPT_ECAPACITY) fill_result(c, out);
    if (rc == ADEPT_OK) rc = rc2;
  }
  return rc;
}

// ---- instrumentation ------------------------------------------------------------------------
uint64_t adept_instr_lines(const adept_ctx *c) { return (c && c->cfg.instrument) ? c->plan.lines_per_kind : 0; }
uint64_t adept_instr_slots(const adept_ctx *c) { return (c && c->cfg.instrument) ? c->plan.slots_per_kind : 0; }

int adept_read_counters(adept_ctx *c, uint64_t *field_rw, uint32_t *lines, uint32_t *slots) {
  if (!c) return ADEPT_EINVAL;
  if (!c->cfg.instrument) return fail(c, ADEPT_ESTATE, "adept_read_counters: context was not created with instrument = 1");
  const Plan &pl = c->plan;
  CU(c, cudaStreamSynchronize(c->stream));
  if (field_rw)
    CU(c, cudaMemcpy(field_rw, c->ws + pl.instr_rw, 3 * kNumFields * 2 * sizeof(uint64_t), cudaMemcpyDeviceToHost));
  for (int k = 0; k < 3; ++k) {
    if (lines)
      CU(c, cudaMemcpy(lines + size_t(k) * pl.lines_per_kind, c->ws + pl.instr_lines[k], pl.lines_per_kind * 4,
                       cudaMemcpyDeviceToHost));
    if (slots)
      CU(c, cudaMemcpy(slots + size_t(k) * pl.slots_per_kind, c->ws + pl.instr_slots[k], pl.slots_per_kind * 4,
                       cudaMemcpyDeviceToHost));
  }
  return ADEPT_OK;
}

int adept_timing_sections(void) {
#ifdef ADEPT_TIMING_SECTIONS
  return 1;
#else
  return 0;
#endif
}

int adept_read_sections(adept_ctx *c, uint64_t *cycles) {
  if (!c || !cycles) return c ? fail(c, ADEPT_EINVAL, "adept_read_sections: cycles is NULL") : ADEPT_EINVAL;
  const int rc = fetch_ctl(c, true);
  if (rc != ADEPT_OK && rc != ADEPT_ECAPACITY) return rc;
  const unsigned long long *s = reinterpret_cast<const unsigned long long *>(c->pinned + kCtlHeaderBytes) +
                                (size_t(2) * c->geo.n_layers + 1);
  for (int i = 0; i < kNumSections; ++i) cycles[i] = s[i];
  return rc;
}

uint32_t adept_launch_index(const adept_ctx *c) { return c ? c->launch_index : 0u; }

int adept_set_launch_index(adept_ctx *c, uint32_t index) {
  if (!c || index >= kLaunchWrap) return ADEPT_EINVAL;
  c->launch_index = index;
  // the restored workspace may hold another population than the one last seen: re-read the live count
  // (it picks the CTA shape of the next launches)
  const int rc = fetch_ctl(c, false);
  return rc == ADEPT_ECAPACITY ? ADEPT_OK : rc;
}

uint64_t adept_field_offset_kind(int32_t layout, uint32_t kind, uint32_t capacity, uint32_t slot, uint32_t field) {
  if (kind > 2u) return UINT64_MAX;
  if (layout != ADEPT_HC16) return adept_field_offset(layout, capacity, slot, field);
  if (field >= uint32_t(kNumFields) || capacity == 0) return UINT64_MAX;
  const size_t cap = (size_t(capacity) + 127) / 128 * 128;
  if (slot >= cap) return UINT64_MAX;
  return 4 * Mapping<L_HC16>::index(cap, slot, int(field), int(kind));
}

uint64_t adept_field_offset(int32_t layout, uint32_t capacity, uint32_t slot, uint32_t field) {
  if (field >= uint32_t(kNumFields) || capacity == 0) return UINT64_MAX;
  const size_t cap = (size_t(capacity) + 127) / 128 * 128;
  if (slot >= cap) return UINT64_MAX;
  switch (layout) {
    case ADEPT_AOS: return 4 * Mapping<L_AOS>::index(cap, slot, int(field));
    case ADEPT_SOA: return 4 * Mapping<L_SOA>::index(cap, slot, int(field));
    case ADEPT_AOSOA32: return 4 * Mapping<L_AOSOA32>::index(cap, slot, int(field));
    case ADEPT_AOSOA64: return 4 * Mapping<L_AOSOA64>::index(cap, slot, int(field));
    case ADEPT_SOA16: return 4 * Mapping<L_SOA16>::index(cap, slot, int(field));
    case ADEPT_AOSOA16: return 4 * Mapping<L_AOSOA16>::index(cap, slot, int(field));
    case ADEPT_AOSOA128: return 4 * Mapping<L_AOSOA128>::index(cap, slot, int(field));
    case ADEPT_AOSOA8: return 4 * Mapping<L_AOSOA8>::index(cap, slot, int(field));
    default: return UINT64_MAX;
  }
}

int adept_dev_math(int fn, const void *in, void *out, uint64_t n, void *cuda_stream) {
  if (fn < 0 || fn > 5 || (n && (!in || !out))) return ADEPT_EINVAL;
  if (n == 0) return ADEPT_OK;
  const unsigned grid = unsigned((n + 255) / 256);
  dev_math_kernel<<<grid, 256, 0, static_cast<cudaStream_t>(cuda_stream)>>>(fn, in, out, n);
  return cudaGetLastError() == cudaSuccess ? ADEPT_OK : ADEPT_ECUDA;
}

}  // extern "C"
