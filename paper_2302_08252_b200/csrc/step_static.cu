// adept_step_static (include/adept.h): the transport step for callers that cannot allocate.
//
// Who this is for.  Every other entry point works on a workspace the caller obtains from cudaMalloc (or
// a framework's allocator) and hands to adept_create, which also pins a small host buffer and creates a
// stream and events.  Some callers may do none of that at the moment they need a step: code running
// between a framework's "memory plan is frozen" point and the end of its step (inference servers and
// simulation hosts that reserve all device memory up front and forbid late allocation), plugin hooks
// that are only handed existing buffers and a stream, and code on a latency budget in which
// cudaMalloc / cudaFree -- which may synchronise the whole device -- are not acceptable.  For them this
// file runs the same step kernel as adept_step (the AoSoA-32 layout on the dense double buffer,
// PAPER.md:31, 121, the variant of SURVEY.md §8(a) rows A0-A11 the benchmark reports) with everything
// that normally lives in the workspace -- the control block with the iteration counters, the energy
// tallies, the device copy of the tables and the two record arrays per particle kind -- placed in ONE
// file-scope __device__ array of fixed size.  The caller passes only inputs and outputs.
//
// What that costs.  The array is part of the library image: every GPU on which the library is loaded
// holds kStaticBytes (about 2.7 MiB) from load to process exit, used or not.  Its size fixes the limits
// ADEPT_STATIC_MAX_* of include/adept.h; larger problems are rejected with ADEPT_EINVAL, never
// truncated.  All calls on a device share the array: it keeps the previous call's contents (this file
// clears the control block and tallies at the start of every call; records and tables are overwritten
// before they are read), and two calls that overlap on one GPU -- different host threads, different
// streams -- would race on it.  The entry point therefore holds a process-wide lock and waits for its own
// work before it returns: it is synchronous, and it cannot serve several streams at once.
//
// Address of the array.  In host code the name of a __device__ variable is a host-side handle, not a
// device pointer; passing it to a kernel makes the kernel fault or, on systems where the GPU can reach
// host memory, silently work on the wrong bytes.  The device address is obtained with
// cudaGetSymbolAddress, once per device, with that device current (static_base below), and that pointer
// is what goes into the kernel parameters.  The first call on a device performs this set-up, so it
// should be made outside any stream capture.
//
// Nothing here calls cudaMalloc, cudaMallocHost, cudaFree, a stream/event constructor or any library
// routine that allocates; host-side temporaries are on the stack.
#include <cstdio>
#include <cstring>
#include <mutex>

#include <cuda_runtime.h>

#include "../../include/adept.h"
#include "step_impl.cuh"

namespace adept {
namespace {

constexpr uint32_t kStaticCapacity = ADEPT_STATIC_MAX_TRACKS;   // slots per kind and array, whole tiles
constexpr uint32_t kStaticLayers = ADEPT_STATIC_MAX_LAYERS;
constexpr uint32_t kStaticBins = ADEPT_STATIC_MAX_BINS;
constexpr uint32_t kStaticMaterials = ADEPT_STATIC_MAX_MATERIALS;
static_assert(kStaticCapacity % kGroup == 0, "capacity is a whole number of tiles");

constexpr size_t up256(size_t x) { return (x + 255) / 256 * 256; }
// [control header | tallies per slab + escaped | section clocks of the timing build]
constexpr size_t kCtlBytes = up256(kCtlHeaderBytes + (size_t(2) * kStaticLayers + 1 + kNumSections + 4) * sizeof(unsigned long long));
// [group 0 = gamma | group 1 = e+-][material][node] float4, as adept_create lays them out
constexpr size_t kTableFloats = size_t(2) * kStaticMaterials * (kStaticBins + 1) * 4;
constexpr size_t kTableBytes = up256(kTableFloats * sizeof(float));
constexpr size_t kRecWords = Mapping<L_AOSOA32>::words(kStaticCapacity);   // one record array
constexpr size_t kRecBytes = up256(kRecWords * 4);
constexpr size_t kOffTables = kCtlBytes;
constexpr size_t kOffRecords = kOffTables + kTableBytes;                   // [kind][current / next]
constexpr size_t kStaticBytes = kOffRecords + 6 * kRecBytes;

// The scratch of adept_step_static.  256-byte alignment: the tables are staged by bulk copies
// (16-byte granules) and a record tile by TMA bulk copies of whole AoSoA blocks.
static __device__ __align__(256) unsigned char g_static_scratch[kStaticBytes];

constexpr int kMaxDevices = 64;
struct DeviceSetup {
  unsigned char *base;   // device address of g_static_scratch on this device
  int sms;
  bool ready;
};
DeviceSetup g_setup[kMaxDevices];
std::mutex g_mutex;                       // one call at a time: the array is shared
thread_local char g_error[256] = "";

int fail(int code, const char *what, cudaError_t e = cudaSuccess) {
  if (e != cudaSuccess) std::snprintf(g_error, sizeof g_error, "%s: %s", what, cudaGetErrorString(e));
  else std::snprintf(g_error, sizeof g_error, "%s", what);
  return code;
}
#define CUS(call)                                               \
  do {                                                          \
    cudaError_t e_ = (call);                                    \
    if (e_ != cudaSuccess) return fail(ADEPT_ECUDA, #call, e_); \
  } while (0)

// Set-up of the current device (first call on it): the device address of the array.
int static_base(DeviceSetup **out) {
  int dev = 0;
  CUS(cudaGetDevice(&dev));
  if (dev < 0 || dev >= kMaxDevices) return fail(ADEPT_EINVAL, "adept_step_static: device ordinal beyond 63");
  DeviceSetup &s = g_setup[dev];
  if (!s.ready) {
    void *ptr = nullptr;
    CUS(cudaGetSymbolAddress(&ptr, g_static_scratch));   // NOT &g_static_scratch: that is a host-side stand-in
    if (!ptr) return fail(ADEPT_ECUDA, "cudaGetSymbolAddress returned NULL");
    CUS(cudaDeviceGetAttribute(&s.sms, cudaDevAttrMultiProcessorCount, dev));
    s.base = static_cast<unsigned char *>(ptr);
    s.ready = true;
  }
  *out = &s;
  return ADEPT_OK;
}

// What set_counts_kernel of adept_api.cu does after adept_load_tracks, for a freshly cleared control
// block: launch 0 finds n_in[k] tracks of kind k in array 0.  Device code may name the array directly.
__global__ void static_begin_kernel(uint32_t n0, uint32_t n1, uint32_t n2) {
  Ctl *ctl = reinterpret_cast<Ctl *>(g_static_scratch);
  const uint32_t n[3] = {n0, n1, n2};
  for (int k = 0; k < 3; ++k) {
    ctl->n[0][k] = n[k];
    ctl->n_cur[k] = n[k];
    ctl->slots_used[k] = n[k];
  }
}

// close_kernel of adept_api.cu for the dense scheme: close the last launch, write the summary fields.
__global__ void static_close_kernel(Params p, uint32_t it) {
#ifdef ADEPT_TIMING_SECTIONS
  roll_iterations<false, false>(p.ctl, p.capacity, it, false, int(threadIdx.x), p.sections);
#else
  roll_iterations<false, false>(p.ctl, p.capacity, it, false, int(threadIdx.x));
#endif
}

}  // namespace
}  // namespace adept

using namespace adept;

extern "C" {

const char *adept_step_static_error(void) { return g_error; }

size_t adept_step_static_bytes(void) { return kStaticBytes; }

int adept_step_static(const adept_geometry *g, const adept_tables *t, const adept_track *const tracks_in[3],
                      const uint32_t n_in[3], adept_track *const tracks_out[3], uint32_t out_capacity,
                      uint32_t iterations, void *cuda_stream, adept_result *out) {
  g_error[0] = 0;
  if (!g || !t || !tracks_in || !n_in || !tracks_out || !out) return fail(ADEPT_EINVAL, "adept_step_static: NULL argument");
  if (g->n_layers == 0 || g->n_layers > kStaticLayers) return fail(ADEPT_EINVAL, "adept_step_static: n_layers outside 1 .. ADEPT_STATIC_MAX_LAYERS");
  if (!(g->abs_mm > 0.0f) || !(g->gap_mm > 0.0f) || !(g->half_xy_mm > 0.0f)) return fail(ADEPT_EINVAL, "adept_step_static: non-positive geometry");
  if (t->n_bins == 0 || t->n_bins > kStaticBins) return fail(ADEPT_EINVAL, "adept_step_static: n_bins outside 1 .. ADEPT_STATIC_MAX_BINS");
  if (t->n_materials == 0 || t->n_materials > kStaticMaterials) return fail(ADEPT_EINVAL, "adept_step_static: n_materials outside 1 .. ADEPT_STATIC_MAX_MATERIALS");
  if (t->physics != 0u) return fail(ADEPT_EINVAL, "adept_step_static: only tables.physics = 0 (the scratch array has no room for the extended rules' side arrays)");
  if (!t->data) return fail(ADEPT_EINVAL, "adept_step_static: tables.data is NULL");
  if (g->mat_abs >= t->n_materials || g->mat_gap >= t->n_materials) return fail(ADEPT_EINVAL, "adept_step_static: material index out of range");
  if (!(t->e_cut > 0.0f) || !(t->e_max > t->e_min) || !(t->e_min > 0.0f)) return fail(ADEPT_EINVAL, "adept_step_static: invalid energy grid");
  if (iterations == 0 || iterations > (1u << 20)) return fail(ADEPT_EINVAL, "adept_step_static: iterations outside 1 .. 2^20");
  for (int k = 0; k < 3; ++k) {
    if (n_in[k] > kStaticCapacity) return fail(ADEPT_EINVAL, "adept_step_static: more than ADEPT_STATIC_MAX_TRACKS tracks of one kind");
    if (n_in[k] && !tracks_in[k]) return fail(ADEPT_EINVAL, "adept_step_static: tracks_in[k] is NULL with n_in[k] > 0");
    if (out_capacity && !tracks_out[k]) return fail(ADEPT_EINVAL, "adept_step_static: tracks_out[k] is NULL");
  }

  std::lock_guard<std::mutex> lock(g_mutex);
  DeviceSetup *dev = nullptr;
  int rc = static_base(&dev);
  if (rc != ADEPT_OK) return rc;
  unsigned char *base = dev->base;
  cudaStream_t stream = static_cast<cudaStream_t>(cuda_stream);
  const LayoutOps &ops = kOpsAoSoA32;
  const uint32_t nodes = t->n_bins + 1, n_slabs = 2 * g->n_layers;

  Params p;
  std::memset(&p, 0, sizeof p);
  p.ctl = reinterpret_cast<Ctl *>(base);
  p.tally = reinterpret_cast<unsigned long long *>(base + kCtlHeaderBytes);
  p.sections = p.tally + (size_t(n_slabs) + 1);
  p.tables = reinterpret_cast<const float4 *>(base + kOffTables);
  p.table_bytes = uint32_t(size_t(t->n_materials) * nodes * sizeof(float4));
  p.table_area = p.table_bytes;
  p.nodes = nodes;
  p.ln_e_min = t->ln_e_min; p.inv_dln = t->inv_dln; p.e_cut = t->e_cut; p.e_max = t->e_max;
  p.n_slabs = n_slabs;
  p.abs_mm = g->abs_mm; p.pitch = g->abs_mm + g->gap_mm; p.half_xy = g->half_xy_mm;
  p.mat_abs = g->mat_abs; p.mat_gap = g->mat_gap;
  p.capacity = kStaticCapacity;
  for (int k = 0; k < 3; ++k) {
    uint32_t *r = reinterpret_cast<uint32_t *>(base + kOffRecords + size_t(2 * k) * kRecBytes);
    p.kind[k].rec[0] = r;
    p.kind[k].rec[1] = reinterpret_cast<uint32_t *>(base + kOffRecords + size_t(2 * k + 1) * kRecBytes);
    // never dereferenced by the dense, plain, physics-0 kernels; kept inside the array all the same
    p.kind[k].queue[0] = p.kind[k].queue[1] = p.kind[k].free_ring = r;
    p.kind[k].msc[0] = p.kind[k].msc[1] = reinterpret_cast<float *>(r);
    p.kind[k].instr_lines = p.kind[k].instr_slots = r;
  }
  p.instr_field_rw = reinterpret_cast<unsigned long long *>(base);

  // CTA shape: the 256-thread one (at most 8192 tracks per kind: a small population, device_state.cuh)
  const size_t dyn = step_smem_bytes(S_DENSE, p.table_area, n_slabs, ops.record_words(kGroup), kBlockSmall, ops.sparse_gather, false);
  const int per_sm = ops.step_ctas_per_sm(S_DENSE, 0, 0, kBlockSmall, dyn);
  if (per_sm <= 0) { cudaGetLastError(); return fail(ADEPT_EINVAL, "adept_step_static: step kernel does not fit on an SM with these tables"); }
  const unsigned grid = unsigned(dev->sms * per_sm);

  // tables: [mat][group][qty][node] (host, ABI) -> [group][mat][node]{q0,q1,q2,0}, on the stack
  float packed[kTableFloats];
  std::memset(packed, 0, sizeof packed);
  for (uint32_t m = 0; m < t->n_materials; ++m)
    for (uint32_t grp = 0; grp < 2; ++grp)
      for (uint32_t q = 0; q < 3; ++q)
        for (uint32_t j = 0; j < nodes; ++j)
          packed[((size_t(grp) * t->n_materials + m) * nodes + j) * 4 + q] = t->data[((size_t(m) * 2 + grp) * 3 + q) * nodes + j];

  // the array keeps the last call's contents: counters and tallies must start at zero
  CUS(cudaMemsetAsync(base, 0, kCtlBytes, stream));
  CUS(cudaMemcpyAsync(base + kOffTables, packed, size_t(2) * p.table_bytes, cudaMemcpyHostToDevice, stream));
  for (int k = 0; k < 3; ++k)
    if (n_in[k]) CUS(ops.launch_load(S_DENSE, p, tracks_in[k], nullptr, n_in[k], k, 0u, 0u, 0u, stream));
  static_begin_kernel<<<1, 1, 0, stream>>>(n_in[0], n_in[1], n_in[2]);
  CUS(cudaGetLastError());
  // the records were validated while they were unpacked (preconditions of adept_load_tracks): the step
  // indexes geometry and tallies with them, so look before stepping
  alignas(16) unsigned char host_ctl[kCtlBytes];
  CUS(cudaMemcpyAsync(host_ctl, base, kCtlHeaderBytes, cudaMemcpyDeviceToHost, stream));
  CUS(cudaStreamSynchronize(stream));
  const Ctl *h = reinterpret_cast<const Ctl *>(host_ctl);
  if (h->bad_input) return fail(ADEPT_EINVAL, "adept_step_static: a record breaks the preconditions (vol, step, ekin, dir; see adept_load_tracks)");

  uint32_t it = 0;
  for (uint32_t i = 0; i < iterations; ++i) {
    p.it = it;
    it = next_launch(it);
    CUS(ops.launch_step(S_DENSE, 0, p, kBlockSmall, grid, dyn, stream));
  }
  static_close_kernel<<<1, 32, 0, stream>>>(p, it);
  CUS(cudaGetLastError());
  const size_t n_fetch = kCtlHeaderBytes + (size_t(n_slabs) + 1) * sizeof(unsigned long long);
  CUS(cudaMemcpyAsync(host_ctl, base, n_fetch, cudaMemcpyDeviceToHost, stream));
  CUS(cudaStreamSynchronize(stream));

  adept_counts &c = out->total;
  for (int k = 0; k < 3; ++k) {
    c.live[k] = h->n_cur[k];
    c.steps[k] = h->steps[k];
    c.secondaries[k] = h->secondaries[k];
    c.killed[k] = h->killed[k];
    c.escaped_n[k] = h->escaped_n[k];
    c.slots_used[k] = h->slots_used[k];
  }
  c.iterations = h->iterations;
  c.overflow = h->overflow;
  c.reserved = 0;
  const unsigned long long *fx = reinterpret_cast<const unsigned long long *>(host_ctl + kCtlHeaderBytes);
  out->e_injected = 0.0;
  out->e_escaped = double(fx[n_slabs]) * kTallyUnit;
  if (out->edep_slab)
    for (uint32_t s = 0; s < n_slabs; ++s) out->edep_slab[s] = double(fx[s]) * kTallyUnit;
  if (out->edep_layer)
    for (uint32_t l = 0; l < g->n_layers; ++l)
      out->edep_layer[l] = double(fx[2 * l]) * kTallyUnit + double(fx[2 * l + 1]) * kTallyUnit;
  if (h->overflow) return fail(ADEPT_ECAPACITY, "adept_step_static: more than ADEPT_STATIC_MAX_TRACKS live tracks of one kind");
  for (int k = 0; k < 3; ++k)
    if (h->n_cur[k] > out_capacity) return fail(ADEPT_EINVAL, "adept_step_static: out_capacity too small (counts are filled in, no track was copied)");
  for (int k = 0; k < 3; ++k)
    if (h->n_cur[k]) CUS(ops.launch_read(S_DENSE, p, tracks_out[k], 0u, h->n_cur[k], k, h->parity, stream));
  CUS(cudaStreamSynchronize(stream));
  return ADEPT_OK;
}

}  // extern "C"
