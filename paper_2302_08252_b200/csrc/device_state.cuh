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

#include <cuda.h>  // CUtensorMap

namespace adept {

enum SchemeId : int { S_SPARSE = 0, S_DENSE = 1 };

// The step kernel is built for two CTA shapes: 256 threads (2 groups, 4 CTAs/SM) for small
// populations -- a shower's head and tail, where CTAs must start and finish quickly -- and 1024
// threads (8 groups, 1 CTA/SM) for large ones, where one staged copy of the tables, one set of tally
// bins and one end-of-iteration ticket per SM are worth 3-4 % (adept_api.cu picks per launch).
constexpr int kBlockSmall = 256, kBlockLarge = 1024;
// A CTA is split into groups of kGroup threads.  A group steps one tile of kGroup tracks at a time
// and synchronises only with itself (a named barrier), so that while one group waits -- for its
// tile's output range (a global atomic) or for a straggling warp -- the other groups of the SM keep
// the schedulers busy.  The groups of a CTA share the staged tables and the tally bins.
#ifndef ADEPT_GROUP
#define ADEPT_GROUP 128
#endif
constexpr int kGroup = ADEPT_GROUP;
constexpr int kMaxGroupsPerCta = kBlockLarge / kGroup;
constexpr int kWarpsPerGroup = kGroup / 32;
static_assert(kGroup == 128, "a group is 4 warps (arrival word: 3 x 9-bit counts + 3-bit ticket; an AoSoA-128 block is one tile)");
// Shared-memory queue (one per group) of tracks parked between the two halves of the step, entry-
// major.  At most kGroup - 1 left over from earlier tiles plus kGroup from the current one.
constexpr int kQueueCap = 2 * kGroup;
// An entry is the 14 record words, the pending interaction packed into the three top bits of the step
// word (steps stay below 2^21, rule S31), and for the sparse scheme the slot (+ one pad word): 56 or
// 64 bytes, written and read as 64-bit words (7 or 8 shared-memory instructions, conflict-free).
// With multiple scattering (rule X39) a parked track of the dense scheme also carries its three cold
// words (in the sparse scheme they stay in place, in the side array): 18 words.
__host__ __device__ constexpr int queue_words(int scheme, bool msc = false) { return scheme == S_DENSE ? (msc ? 18 : 14) : 16; }
__host__ __device__ constexpr size_t queue_bytes(int scheme, bool msc = false) { return size_t(kQueueCap) * queue_words(scheme, msc) * 4; }
// One tile of records staged in shared memory per group (record_words(kGroup) words of the layout):
// dense scheme, by TMA bulk / tiled copies of the contiguous tile; sparse scheme, by per-thread
// asynchronous copies (cp.async) of the records the group's list entries name, followed by two words
// per thread -- the slot of the gathered record and the thread's list entry for the tile after it,
// which also arrives by cp.async.  Both schemes fetch one tile ahead of the tile being stepped.
// `gather`: the layout keeps a record's words in 16-byte pieces (layout.cuh Mapping<L>::kSparseGather);
// the word-by-word layouts load their records directly and stage nothing (measured: 14 four-byte
// asynchronous copies per record and the L1 capacity given up for the staging buffer cost them more
// than the latency they hide -- DESIGN.md §10).
__host__ __device__ constexpr size_t in_buf_bytes(int scheme, size_t tile_words, bool gather) {
  // sparse, direct loads: only the two stash words per thread (list entries of the next two tiles)
  return scheme == S_DENSE ? tile_words * 4 : (gather ? tile_words * 4 : 0) + 2 * size_t(kGroup) * 4;
}
// Tally bins of a CTA: per slab (+ one bin for the energy carried out of the calorimeter) a 64-bit
// fixed-point sum kept as two 32-bit limbs, [lo limbs][hi limbs].
__host__ __device__ constexpr size_t bins_bytes(uint32_t n_slabs) { return ((size_t(n_slabs) + 1) * 8 + 15) / 16 * 16; }
// Dynamic shared memory of the step kernel: [tables of one particle group][bins][per group: staged tile, queue]
// (the per-group part starts on a 128-byte boundary: what a tiled TMA copy needs of its destination)
__host__ __device__ constexpr size_t units_offset(size_t table_bytes, uint32_t n_slabs) {
  return (table_bytes + bins_bytes(n_slabs) + 127) / 128 * 128;
}
__host__ __device__ constexpr size_t step_smem_bytes(int scheme, size_t table_bytes, uint32_t n_slabs, size_t tile_words,
                                                     int threads, bool gather, bool msc = false) {
  return units_offset(table_bytes, n_slabs) + size_t(threads / kGroup) * (in_buf_bytes(scheme, tile_words, gather) + queue_bytes(scheme, msc));
}

// Energy tallies (rule M7: sums of fp32 terms) are accumulated in 64-bit fixed point, unit
// 2^-32 MeV: every term is rounded to the unit once (absolute error <= 2^-33 MeV = 1.2e-10 MeV),
// after which the additions are exact and therefore independent of the order in which threads,
// warps and CTAs arrive.  Range 2^32 MeV (4.3e3 TeV) per slab.
constexpr double kTallyUnit = 1.0 / 4294967296.0;

// Iteration control without a "last CTA".  Every launch carries its
// launch index `it` (Params::it, counted by the host).  The per-iteration counters are kept three
// deep, indexed by launch index modulo 3: launch `it` reads n[it % 3] (what is alive), accumulates its
// outputs into n[(it + 1) % 3] and its statistics into alive/esc[it % 3]; nobody touches the third
// buffer during the launch, which is where the first warp of CTA 0 works: at the start of launch `it`
// it closes launch it - 1 (adds its statistics to the cumulative counters, then clears its buffers for
// launch it + 2) and opens launch `it`.  No CTA has to be the last one, so the end of an iteration is
// not a link in the chain of round trips a small population's iteration consists of.
// The host reads the control block only through close_kernel (adept_api.cu), which closes whatever
// is open and writes the summary fields n_cur / parity.
// Launch indices count modulo kLaunchWrap, a multiple of 6 just below 2^32, so that `it % 3` and
// `it & 1` stay continuous when the counter wraps (after 4e9 launches).
constexpr uint32_t kLaunchWrap = 4294967292u;
static_assert(kLaunchWrap % 6u == 0u, "parity and buffer index must survive the wrap");
__host__ __device__ constexpr uint32_t next_launch(uint32_t it) { return it + 1u == kLaunchWrap ? 0u : it + 1u; }

struct Ctl {
  uint32_t n[3][4];       // dense: tracks in the array; sparse: length of the slot list -- by launch index % 3
  uint32_t alive[3][4];   // parents that survived the launch, per kind
  uint32_t esc[3][4];     // parents that left the calorimeter in the launch, per kind
  // sparse scheme with ADEPT_FLAG_RECYCLE_SLOTS: ring of freed slots per kind (KindStorage::free_ring).
  // Monotonic counters, ring index = counter % capacity.  Slots freed in launch `it` are pushed at
  // `free_tail` and become allocatable in launch it + 1: ring_tail[it % 3] is the tail as it was when
  // launch `it` began (pushes of launch `it` are also counted into ring_tail[(it + 1) % 3], to which
  // CTA 0 adds ring_tail[it % 3] itself), and pops take positions below it, so pushes and pops never
  // meet inside a launch.  A pop that runs past it gives the excess back (free_head never passes it).
  uint32_t ring_tail[3][4];
  uint32_t slot_top[4];   // sparse: bump allocator of never-recycled slots (rule S30)
  uint32_t free_head[4], free_tail[4];
  uint32_t overflow;      // sticky
  uint32_t bad_input;     // set by load_kernel when a record breaks the preconditions of adept_load_tracks
  uint32_t closed;        // launches closed so far (= the index of the next launch once everything is closed)
  uint32_t parity;        // summary (close_kernel): which array / list is "current" for the next launch
  uint32_t n_cur[4];      // summary (close_kernel): live tracks per kind
  unsigned long long steps[3], secondaries[3], killed[3], escaped_n[3], slots_used[3];
  unsigned long long iterations;
  // unsigned long long tally[n_slabs + 1] follows at byte kCtlHeaderBytes: fixed-point energy
  // deposit per slab, then the energy carried out of the calorimeter
};
constexpr size_t kCtlHeaderBytes = 512;
static_assert(sizeof(Ctl) <= kCtlHeaderBytes, "control block header");

struct KindStorage {
  uint32_t *rec[2];    // dense: current/next arrays by parity; sparse: rec[0] only
  uint32_t *queue[2];  // sparse: slot lists by parity
  uint32_t *free_ring;    // sparse + slot recycling: [capacity] freed slots (Ctl::free_head / free_tail)
  // physics 2 (rule X39), e- and e+ only: the three multiple-scattering words of a track -- the paper's
  // cold fields InitialRange, DynamicRangeFactor, TlimitMin -- as a side array
  // [3][capacity] next to the records, addressed like them (dense: by parity; sparse: msc[0], by slot)
  float *msc[2];
  uint32_t *instr_lines;  // instrumented build: per 128-B line of this kind's record storage
  uint32_t *instr_slots;  // instrumented build: per slot (dense: 2 * capacity)
};

struct Params {
  Ctl *ctl;
  unsigned long long *tally; // [n_slabs + 1] fixed point, right after the control header
  unsigned long long *sections;  // [kNumSections] warp-cycles per kernel section (timing build; after the tallies)
  const float4 *tables;      // [group][material][node] {q0, q1, q2, 0}; group 0 = gamma, 1 = e+-
  uint32_t table_bytes;      // bytes of ONE group, multiple of 16
  uint32_t table_area;       // shared-memory bytes of the staged tables: one group, or (extended physics) the
                             // e+- group followed by the e+ extras
  uint32_t nodes;            // n_bins + 1
  float ln_e_min, inv_dln, e_cut, e_max;
  uint32_t n_slabs;
  float abs_mm, pitch, half_xy;
  uint32_t mat_abs, mat_gap;
  uint32_t capacity;         // slots per kind (multiple of 128)
  uint32_t recycle;          // sparse scheme: 1 = freed slots are reused (ADEPT_FLAG_RECYCLE_SLOTS)
  uint32_t physics;          // adept_tables.physics: 1 = extended rules X36-X38, 2 = also X39 (multiple scattering)
  uint32_t it;               // index of this launch (counted by the host; see Ctl)
  KindStorage kind[3];
  unsigned long long *instr_field_rw;  // [3][14][2], instrumented build
  // SoA and AoS layouts, dense scheme: tensor maps of the record buffers, [kind][parity] (see
  // prefetch_tile in step_impl.cuh)
  alignas(64) CUtensorMap tile_map[3][2];
};

}  // namespace adept
