// Device-resident state of a context and the parameter block passed to every kernel.
//
// the sparse single buffer is "one sparse array of tracks per particle type" plus "two
// lists of integers ... managing the track slots of the current and subsequent transport
// iteration"; the dense double buffer is "two dense arrays of track structures, one
// for the currently active particles and one for the particles active in the next iteration".
// Both are carved out of the caller's workspace; `Ctl` holds their counters so that an iteration
// needs no host round trip.
#pragma once
#include <cstddef>
#include <cstdint>

namespace adept {

enum SchemeId : int { S_SPARSE = 0, S_DENSE = 1 };

constexpr int kBlock = 256;  // threads per CTA of the step kernel = tracks per tile
// Shared-memory queue of tracks parked between the two halves of the step: 14 record words + the
// pending interaction (+ the slot, sparse scheme only), field-major.  At most kBlock - 1 left over
// from earlier tiles plus kBlock from the current one.
constexpr int kQueueCap = 2 * kBlock;
__host__ __device__ constexpr int queue_words(int scheme) { return scheme == S_DENSE ? 15 : 16; }
__host__ __device__ constexpr size_t queue_bytes(int scheme) { return size_t(kQueueCap) * queue_words(scheme) * 4; }
// Dense scheme: one tile staged in shared memory by TMA (record_words(kBlock) words of the layout).
__host__ __device__ constexpr size_t in_buf_bytes(int scheme, size_t tile_words) {
  return scheme == S_DENSE ? tile_words * 4 : 0;
}

struct Ctl {
  // dense: tracks in the current / next array.  sparse: length of the current / next slot list.
  uint32_t n_cur[4];
  uint32_t n_next[4];
  uint32_t slot_top[4];  // sparse: bump allocator of never-recycled slots (rule S30)
  uint32_t parity;       // which array / list is "current"
  uint32_t overflow;     // sticky
  uint32_t done_ctas;    // ticket counter: the last CTA of a step kernel ends the iteration
  uint32_t pad0;
  uint32_t it_alive[4];    // this iteration: parents that survive, per kind (reset at iteration end)
  uint32_t it_escaped[4];  // this iteration: parents that left the calorimeter, per kind
  unsigned long long steps[3], secondaries[3], killed[3], escaped_n[3], slots_used[3];
  unsigned long long iterations;
  double e_escaped;
  unsigned long long pad1[2];
  // double edep[n_slabs] follows at byte kCtlHeaderBytes
};
constexpr size_t kCtlHeaderBytes = 256;
static_assert(sizeof(Ctl) <= kCtlHeaderBytes, "control block header");

struct KindStorage {
  uint32_t *rec[2];    // dense: current/next arrays by parity; sparse: rec[0] only
  uint32_t *queue[2];  // sparse: slot lists by parity
  uint32_t *instr_lines;  // instrumented build: per 128-B line of this kind's record storage
  uint32_t *instr_slots;  // instrumented build: per slot (dense: 2 * capacity)
};

struct Params {
  Ctl *ctl;
  double *edep;              // [n_slabs], right after the control header
  const float4 *tables;      // [group][material][node] {q0, q1, q2, 0}; group 0 = gamma, 1 = e+-
  uint32_t table_bytes;      // bytes of ONE group, multiple of 16
  uint32_t nodes;            // n_bins + 1
  float ln_e_min, inv_dln, e_cut;
  uint32_t n_slabs;
  float abs_mm, pitch, half_xy;
  uint32_t mat_abs, mat_gap;
  uint32_t capacity;         // slots per kind (multiple of 32)
  KindStorage kind[3];
  unsigned long long *instr_field_rw;  // [3][14][2], instrumented build
};

}  // namespace adept
