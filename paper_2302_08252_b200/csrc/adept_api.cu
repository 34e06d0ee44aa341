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
  size_t rec[3], queue[3][2];
  size_t instr_rw, instr_lines[3], instr_slots[3];
  size_t total;
  uint32_t capacity;       // rounded up to a multiple of 32
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
    default: return nullptr;
  }
}

static bool make_plan(const adept_geometry *g, const adept_tables *t, const adept_config *c, Plan &pl) {
  if (!g || !t || !c) return false;
  const LayoutOps *ops = ops_for(c->layout);
  if (!ops) return false;
  if (c->scheme != ADEPT_SPARSE_SINGLE && c->scheme != ADEPT_DENSE_DOUBLE) return false;
  if (g->n_layers == 0 || g->n_layers > 2048) return false;
  if (t->n_bins == 0 || t->n_bins > 4096 || t->n_materials == 0 || t->n_materials > 8) return false;
  if (c->capacity_per_kind == 0 || c->capacity_per_kind > (1u << 30)) return false;
  pl.capacity = (c->capacity_per_kind + 31u) / 32u * 32u;
  pl.nbuf = (c->scheme == ADEPT_DENSE_DOUBLE) ? 2 : 1;
  pl.rec_words = ops->record_words(pl.capacity);
  pl.table_bytes = size_t(t->n_materials) * 2 * (t->n_bins + 1) * sizeof(float4);
  pl.stage_records = std::min<uint32_t>(pl.capacity, kStageRecords);
  size_t off = 0;
  pl.ctl = off; off = align_up(off + kCtlHeaderBytes + size_t(2) * g->n_layers * sizeof(double));
  pl.tables = off; off = align_up(off + pl.table_bytes);
  pl.stage = off; off = align_up(off + size_t(pl.stage_records) * kStageRecordBytes);
  pl.stage_slots = off; off = align_up(off + size_t(pl.stage_records) * 4);
  for (int k = 0; k < 3; ++k) {
    pl.rec[k] = off; off = align_up(off + pl.rec_words * 4 * pl.nbuf);
    for (int q = 0; q < 2; ++q) {
      pl.queue[k][q] = off;
      if (c->scheme == ADEPT_SPARSE_SINGLE) off = align_up(off + size_t(pl.capacity) * 4);
    }
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
  unsigned grid;
  size_t dyn_smem;
  unsigned char *ws;
  unsigned char *pinned;  // kCtlHeaderBytes + edep
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

// copy control block (+ edep) to pinned memory and wait
int fetch_ctl(adept_ctx *c, bool with_edep) {
  const size_t n = with_edep ? c->pinned_bytes : kCtlHeaderBytes;
  CU(c, cudaMemcpyAsync(c->pinned, c->ws + c->plan.ctl, n, cudaMemcpyDeviceToHost, c->stream));
  CU(c, cudaStreamSynchronize(c->stream));
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
  out->e_escaped = h->e_escaped;
  const double *edep = reinterpret_cast<const double *>(c->pinned + kCtlHeaderBytes);
  if (out->edep_slab) std::memcpy(out->edep_slab, edep, size_t(2) * c->geo.n_layers * sizeof(double));
  if (out->edep_layer)
    for (uint32_t l = 0; l < c->geo.n_layers; ++l) out->edep_layer[l] = edep[2 * l] + edep[2 * l + 1];
}

// write n_cur / slot_top / slots_used of one kind after a host-driven append
__global__ void set_counts_kernel(Ctl *ctl, int kind, uint32_t n_cur, uint32_t slot_top, unsigned long long used) {
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
    default: {
      float s, c;
      sincos2pi(static_cast<const float *>(in)[i], s, c);
      static_cast<float2 *>(out)[i] = make_float2(s, c);
    }
  }
}

}  // namespace
