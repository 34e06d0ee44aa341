/* adept.h — C ABI of the B200-native AdePT transport step (arXiv 2302.08252 hot path).
 *
 * What the library computes.  The paper keeps, per particle type (e-, e+, gamma), "a list of
 * active particle tracks"; every iteration runs one transport pass per type, and survivors and
 * secondaries go to next-iteration storage (§2).  Two containers are described: the
 * sparse single buffer with two integer slot lists (Fig. 1a) and the dense double
 * buffer (Fig. 1b).  The record layout is switched at compile time between AoS, SoA
 * and AoSoA-n.  The result of a run is "the energy deposit in the
 * detector's layers" of a stack of "50 alternating box-shaped layers of absorber and gap material"
 * (§4).  The four calls create / inject / step / run are named by
 * BASELINE.json:north_star; what one step computes is DESIGN.md §3 (rules R1-R6, M7-M11, T12-T15,
 * S16-S32), the simplified analytic physics BASELINE.json prescribes.
 *
 * Conventions.
 *  - Every function returns ADEPT_OK (0) or a negative adept_status; nothing throws across the ABI.
 *  - "host" pointers are ordinary CPU memory, read or written during the call only (copied, never
 *    kept).  "device" pointers are CUDA global memory of the current device.
 *  - The caller owns everything it passes, including the device workspace, which must stay alive
 *    and untouched (except as noted under "Workspace") until adept_destroy.  The library allocates
 *    no device memory; it keeps a small pinned host buffer for count read-back.
 *  - All device work is enqueued on config.cuda_stream (a cudaStream_t, NULL = legacy default
 *    stream).  Calls that return data synchronise that stream; adept_step(ctx, NULL) does not.
 *  - A context is not thread-safe.  Units: MeV, mm.  Particle kinds: 0 = e-, 1 = e+, 2 = gamma.
 *  - Capacity overflow: a full buffer/queue sets a device flag, the step completes without any
 *    out-of-bounds write (excess tracks are dropped), and the next synchronising call returns
 *    ADEPT_ECAPACITY; afterwards only adept_reset / adept_destroy are accepted.  The same flag is
 *    raised if an energy tally leaves its 64-bit fixed-point range (2^32 MeV in one slab).
 *
 * Workspace.  The workspace holds the complete device state of a context (control block, tables,
 * track buffers, queues, tallies).  A byte copy of it taken while no call is in flight, together with
 * adept_launch_index() at that moment, may be written back later -- followed by
 * adept_set_launch_index() -- to rewind the context (bench.py restores a pristine copy between timed
 * steps this way).  The launch index is the one piece of iteration state the host holds: the device keeps
 * its per-iteration counters three deep, indexed by it, so that no thread block has to close an
 * iteration.
 */
#ifndef ADEPT_B200_H
#define ADEPT_B200_H

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct adept_ctx adept_ctx; /* opaque, host object */

typedef enum {
  ADEPT_OK = 0,
  ADEPT_EINVAL = -1,    /* bad argument; nothing was changed */
  ADEPT_ECAPACITY = -2, /* a track buffer or queue overflowed (see above) */
  ADEPT_ECUDA = -3,     /* a CUDA call failed; adept_last_error() has the text */
  ADEPT_ESTATE = -4     /* call not allowed in the context's current state */
} adept_status;

/* Record layout in device memory ("AoS", "SoA", "AoSoA-n" with n = 8, 16, 32, 64 or 128
 * lanes; AoSoA64 on the dense double buffer was the paper's fastest variant), and "SoA16": SoA of
 * 16-byte field groups {pos.xyz, dir.x} {dir.y, dir.z, ekin, nial.0} {nial.1, nial.2, vol, id_lo}
 * {id_hi, step} -- the hot/cold grouping the paper's conclusion points to. */
typedef enum { ADEPT_AOS = 0, ADEPT_SOA = 1, ADEPT_AOSOA32 = 2, ADEPT_AOSOA64 = 3, ADEPT_SOA16 = 4,
               ADEPT_AOSOA16 = 5, ADEPT_AOSOA128 = 6, ADEPT_HC16 = 7, ADEPT_AOSOA8 = 8 } adept_layout;
/* ADEPT_HC16: hot/cold split with per-kind grouping ("a separation of hot and cold data
 * would be a first step", "different layouts per particle type"): the SoA16 geometry with the words of a
 * record regrouped, per particle kind, into two vectors the step rewrites every time ({pos, step} and
 * gamma: {nial.0-2, vol} / e+-: {ekin, nial.0, nial.1, vol}), one it only reads unless an interaction
 * happens (gamma: {dir, ekin} / e+-: {dir, nial.2}) and the cold {id_lo, id_hi}.  The sparse single
 * buffer then rewrites 32 bytes of a record per step instead of 56-64. */
/* Track container (PAPER.md:29 / PAPER.md:31). */
typedef enum { ADEPT_SPARSE_SINGLE = 0, ADEPT_DENSE_DOUBLE = 1 } adept_scheme;

/* Slab calorimeter: layer L = absorber slab 2L then gap slab 2L+1 along +z,
 * starting at z = 0; transverse box |x|,|y| <= half_xy_mm; outside is vacuum (escape). */
typedef struct {
  uint32_t n_layers;         /* 1 .. 2048 */
  float abs_mm, gap_mm;      /* slab thicknesses, > 0 */
  float half_xy_mm;          /* > 0 */
  uint32_t mat_abs, mat_gap; /* material index of each slab type, < n_materials */
} adept_geometry;

/* fp32 log-grid tables (DESIGN.md rules T12-T14).  data is a HOST array
 * [n_materials][group 2][qty 3][n_bins+1]: group 0 = gamma {pair, Compton, photoelectric} [1/mm];
 * group 1 = e+- {bremsstrahlung [1/mm], stopping power [MeV/mm], range [mm]}.  Copied at create. */
typedef struct {
  uint32_t n_bins, n_materials;
  float e_min, e_max;      /* grid end points [MeV] */
  float ln_e_min, inv_dln; /* fl32(ln e_min), fl32(n_bins / ln(e_max/e_min)) */
  float e_cut;             /* production = tracking cut [MeV] */
  const float *data;       /* host */
  /* Extended physics (DESIGN.md rules X35-X39).  physics = 0: the rules
   * S16-S32 only (data_x ignored).  physics = 1: e+- also produce delta rays (the 1/T^2 term common to
   * Moller and Bhabha scattering, on nial[1]), e+ also annihilate in flight (on nial[2]), and the
   * Compton energy fraction is sampled from the full Klein-Nishina distribution.  physics = 2: e+- are
   * also deflected by multiple scattering, which limits their step by max(DynamicRangeFactor *
   * InitialRange, TlimitMin) -- the paper's three cold track fields, kept per track
   * in a side array of the workspace, not in the 14-word record (a track handed in through the ABI
   * starts uninitialised, like a new one).  data_x is a HOST array [n_materials][3][n_bins+1] of
   * {Sigma_delta, Sigma_annihilation, Sigma_transport} [1/mm], and the stopping power / range in `data`
   * must be the ones restricted to losses below the cut.  physics >= 1 is not available in instrumented
   * contexts or with ADEPT_FLAG_RECYCLE_SLOTS (EINVAL). */
  uint32_t physics;
  const float *data_x;     /* host */
} adept_tables;

typedef struct {
  int32_t layout;             /* adept_layout */
  int32_t scheme;             /* adept_scheme */
  uint32_t capacity_per_kind; /* slots per particle kind (dense: per buffer), 1 .. 2^30; rounded up to a
                               * multiple of 128 (one tile) */
  uint32_t batch_primaries;   /* adept_run: 0 = inject everything at once, else batch size */
  uint64_t seed;              /* primary ids, rule R4 */
  void *workspace;            /* device, 256-byte aligned, >= adept_workspace_bytes() */
  size_t workspace_bytes;
  void *cuda_stream;          /* cudaStream_t */
  uint32_t instrument;        /* 1 = counting build of the same kernels */
  uint32_t flags;             /* 0 or ADEPT_FLAG_*; unknown bits are rejected */
} adept_config;

/* Sparse single buffer only (ignored by the dense double buffer).  The paper's container hands out
 * slots "atomically" and never reuses one within a batch (2044 dense slots against
 * 45509 sparse ones for the same run) -- that policy is the default (DESIGN.md rule S30).  With this
 * flag the slot of every track that ends is pushed onto a per-kind ring of free slots, and secondaries
 * take slots from the ring (those freed up to the previous iteration) before bump-allocating new
 * ones.  Results are unchanged (slots carry no physics); adept_counts.slots_used
 * then reports the real footprint. */
#define ADEPT_FLAG_RECYCLE_SLOTS 1u

typedef struct { uint32_t kind; float pos[3], dir[3], ekin; } adept_primary; /* 32 B */

/* One track, 14 four-byte words.  nial = number of interaction lengths left
 * ("NumIALeft"); vol = slab index (navigation state); (id_lo,id_hi,step) address the
 * track's Philox-4x32-10 stream (rule R2). */
typedef struct {
  float pos[3], dir[3], ekin, nial[3];
  uint32_t vol, id_lo, id_hi, step;
} adept_track; /* 56 B */

typedef struct {
  uint64_t live[3];        /* tracks alive now, per kind */
  uint64_t steps[3];       /* track-steps taken so far, per kind (rule S28) */
  uint64_t secondaries[3]; /* tracks created so far, per kind of the NEW track */
  uint64_t killed[3];      /* tracks that ended (absorbed, below cut, escaped), per kind */
  uint64_t escaped_n[3];   /* of which left the calorimeter */
  uint64_t slots_used[3];  /* dense: high-water live count; sparse: high-water of the slot allocator */
  uint64_t iterations;     /* iterations in which at least one track was alive */
  uint32_t overflow;       /* 1 after a capacity overflow */
  uint32_t reserved;
} adept_counts;

/* Energies are accumulated on the device in 64-bit fixed point of unit 2^-32 MeV (every fp32 term
 * rounded to the unit once, then exact, order-independent integer sums; range 2^32 MeV per slab) and
 * converted to double here (DESIGN.md §3 reading 33). */
typedef struct {
  adept_counts total;
  double e_injected; /* sum of primary kinetic energies (+ 2 mc^2 per e+), MeV */
  double e_escaped;  /* energy carried out of the calorimeter, MeV */
  double *edep_slab;  /* host, caller buffer of 2*n_layers doubles, or NULL */
  double *edep_layer; /* host, caller buffer of n_layers doubles (slab 2L + slab 2L+1), or NULL */
} adept_result;

/* Bytes of device workspace a context with these parameters needs (0 on invalid arguments).
 * Only geometry.n_layers, tables.n_bins/n_materials and config.layout/scheme/capacity/instrument
 * are read. */
size_t adept_workspace_bytes(const adept_geometry *, const adept_tables *, const adept_config *);

/* Build a context: validates, copies geometry and tables to the workspace, clears all state. */
int adept_create(const adept_geometry *, const adept_tables *, const adept_config *, adept_ctx **out);

/* Add n primaries (host array).  batch_primaries == 0: they become live tracks immediately (ids by
 * rule R4 from a running global index; slab located from pos.z); otherwise they are queued for
 * adept_run.  EINVAL if a primary is outside the calorimeter or its energy outside [e_cut, e_max]. */
int adept_inject(adept_ctx *, const adept_primary *primaries, uint64_t n);

/* Rule R4: primary ids (hence random streams) derive from a running global primary index that
 * starts at 0 at create/reset.  A caller that simulates only the slice [lo, hi) of a longer primary
 * list (one rank of a multi-GPU run; events are independent) sets the index to lo
 * before injecting, so that every primary keeps the id it has in the unsliced run and the per-rank
 * tallies add up to the single-GPU result.  ESTATE while queued primaries (batch mode) are pending. */
int adept_set_primary_index(adept_ctx *, uint64_t next_index);

/* One iteration: every live track of every kind takes one step (DESIGN.md rules S16-S28).
 * out == NULL: enqueue only.  out != NULL: synchronise and report the counts after the step. */
int adept_step(adept_ctx *, adept_counts *out);

/* Iterate until no track is alive (and no primary is pending), or max_iterations (0 = no limit)
 * iterations were done in this call -- iterations as adept_counts.iterations counts them: those in
 * which at least one track was alive.  The limit is tested before a pending batch is injected, so no
 * un-stepped batch is left behind.  Fills *out (tallies are cumulative since create/reset). */
int adept_run(adept_ctx *, uint64_t max_iterations, adept_result *out);

/* Fill *out with the current tallies without stepping (synchronises). */
int adept_get_result(adept_ctx *, adept_result *out);

/* Append n tracks (host array, 56-byte records) to kind's live set.  slots (host, n entries) is
 * used by the sparse scheme only: slot of each track, all distinct, free and < capacity (slots are
 * handed out by a bump allocator, rule S30: the free ones are those at or above its top, i.e. above
 * every slot used so far); NULL = next free slots.  The queue order is the array order.
 * Preconditions on every record (the step indexes geometry and tallies by vol, packs flags into the
 * top bits of step, and divides by the direction cosines): vol < 2*n_layers; step < 2^20;
 * e_cut <= ekin <= e_max (an e+ may also have 0 <= ekin < e_cut: it annihilates at its next step,
 * rule S17); pos and dir finite, dir not the zero vector; nial not NaN.
 * EINVAL if a slot or a record breaks these (records are checked on the device while they are
 * unpacked, i.e. after the transfer): the live set and its counts are unchanged then, but storage beyond
 * the live set (free slots, the tail of the dense array) may hold the records that were valid. */
int adept_load_tracks(adept_ctx *, uint32_t kind, const adept_track *tracks, uint64_t n,
                      const uint32_t *slots);

/* Copy kind's live tracks to a host array of cap records (buffer order: unspecified, rule S29).
 * *n receives the live count; ECAPACITY-free: if *n > cap nothing is copied and EINVAL returns. */
int adept_read_tracks(adept_ctx *, uint32_t kind, adept_track *out, uint64_t cap, uint64_t *n);

/* Instrumented contexts only (config.instrument = 1), all host buffers, any may be NULL:
 *  field_rw[3][14][2]  u64: per kind, per record word, {reads, writes} done by the step kernel
 *                      through the layout accessor (Fig. 5);
 *  lines[3][n_lines]   u32: accesses per 128-byte line of each kind's record storage, where
 *                      n_lines = adept_instr_lines(ctx) (PAPER.md:131, 135 heatmap, row = cache line);
 *  slots[3][n_slots]   u32: accesses per track slot, n_slots = adept_instr_slots(ctx). */
int adept_read_counters(adept_ctx *, uint64_t *field_rw, uint32_t *lines, uint32_t *slots);
uint64_t adept_instr_lines(const adept_ctx *);
uint64_t adept_instr_slots(const adept_ctx *);

/* Timing variant of the library (built with -DADEPT_TIMING_SECTIONS as libadept_b200_timing.so;
 * BASELINE.json configs[3]: "each scheme reports step plus slot-allocation/compaction time").
 * Allocation and compaction are fused into the step kernel, so the
 * variant brackets the sections of every tile with the SM clock and sums, over lane 0 of every
 * warp, the cycles spent in each: cycles[0] other (prologue, table staging, tally flush),
 * [1] A1 record load, [2] A2-A7 move half, [3] A8 interact half, [4] A9 allocation (ballots, arrival
 * word, range/slot reservation, group barrier, ranks), [5] A10 stores (records, slot lists, parked
 * queue); [6] nanoseconds from the first thread block's start to the last one's end, summed over the
 * launches; [7] unused.  Cumulative since create/reset.  adept_timing_sections() returns 1 in
 * the timing variant, 0 otherwise (all cycles then read 0).  cycles: host, ADEPT_N_SECTIONS entries. */
#define ADEPT_N_SECTIONS 8
int adept_timing_sections(void);
int adept_read_sections(adept_ctx *, uint64_t *cycles);

/* Byte offset of word `field` (0..13: pos xyz, dir xyz, ekin, nial 0-2, vol, id_lo, id_hi, step) of
 * slot `slot` inside one record buffer of `capacity` slots under `layout` (Fig. 3:
 * where each field is placed).  Pure host arithmetic; UINT64_MAX on invalid arguments. */
uint64_t adept_field_offset(int32_t layout, uint32_t capacity, uint32_t slot, uint32_t field);
/* The same for layouts whose placement depends on the particle kind (ADEPT_HC16; for the others `kind`
 * only has to be valid).  adept_field_offset itself returns UINT64_MAX for ADEPT_HC16. */
uint64_t adept_field_offset_kind(int32_t layout, uint32_t kind, uint32_t capacity, uint32_t slot, uint32_t field);

/* Number of step launches enqueued since create/reset (see "Workspace"); set: only together with a
 * restored workspace copy taken at that index. */
uint32_t adept_launch_index(const adept_ctx *);
int adept_set_launch_index(adept_ctx *, uint32_t index);
/* Only device state is rewound by writing a workspace copy back: primaries queued for adept_run,
 * e_injected and the primary index are host state and stay as they are.  The live count the host uses to
 * pick the CTA shape is refreshed from the device at the next call that synchronises. */

/* Drop all tracks, pending primaries and tallies; keeps geometry, tables and configuration. */
int adept_reset(adept_ctx *);
int adept_destroy(adept_ctx *);
/* Text of the last error of this context ("" if none).  ctx may be NULL: last create error. */
const char *adept_last_error(const adept_ctx *);

/* The step for callers that cannot allocate (csrc/step_static.cu).
 *
 * Every call above needs a workspace from cudaMalloc (or a framework allocator), and adept_create also
 * pins host memory and creates a stream and events.  Some callers cannot do that when they need a step:
 * hosts that reserve all device memory at start-up and forbid allocation afterwards, plugin hooks that
 * receive only existing buffers and a stream, and code on a latency budget that cannot afford
 * cudaMalloc / cudaFree (either may synchronise the whole device).  adept_step_static runs the same
 * step kernel (AoSoA-32 records, dense double buffer: PAPER.md:31, 121; rules S16-S32) and keeps
 * everything the workspace would hold -- control block, tallies, device tables, both record arrays of
 * each kind -- in one fixed __device__ array inside the library.  It calls no cudaMalloc, cudaMallocHost,
 * cudaFree, stream/event constructor or allocating library routine.
 *
 * Limits (the price of the fixed array, which occupies adept_step_static_bytes() ~ 2.7 MiB on every GPU
 * that loads the library, from load to process exit): at most ADEPT_STATIC_MAX_TRACKS tracks per kind,
 * before and after every iteration; ADEPT_STATIC_MAX_LAYERS layers; ADEPT_STATIC_MAX_BINS table bins;
 * ADEPT_STATIC_MAX_MATERIALS materials; tables.physics = 0 only.  Anything larger returns ADEPT_EINVAL
 * before any work is enqueued (a population that outgrows the array while stepping: ADEPT_ECAPACITY,
 * counts filled in, no tracks copied).
 *
 * Arguments.  geometry, tables: host, as for adept_create (tables.data is copied during the call).
 * tracks_in[k]: DEVICE array of n_in[k] records of kind k (may be NULL when n_in[k] = 0); the
 * preconditions of adept_load_tracks apply (EINVAL otherwise, nothing stepped).  tracks_out[k]: DEVICE
 * array with room for out_capacity records; on return its first out->total.live[k] records are the
 * kind-k tracks alive after `iterations` (>= 1) iterations, in unspecified order (rule S29).  If a kind
 * has more than out_capacity live tracks: EINVAL, counts filled in, no track copied.  *out: counts and
 * tallies of these iterations alone (e_injected is 0: the call does not know what was injected);
 * edep_slab / edep_layer as in adept_result.  n_in, tracks_in, tracks_out: host arrays of 3 entries.
 * cuda_stream: all work is enqueued there; the call returns after it has completed.
 *
 * Sharing.  All calls on a device use the one array.  It keeps the last call's contents; the call
 * clears what must start at zero (counters, tallies) itself.  Two calls overlapping on one GPU would
 * race on it, so the entry point holds a process-wide lock and waits for its own work: it cannot run
 * concurrently on several streams.  The first call on each device looks up the array's device address
 * (one-time set-up); make that first call outside any stream capture.
 * adept_step_static_error(): text of the calling thread's last failure ("" if none). */
#define ADEPT_STATIC_MAX_TRACKS 8192u
#define ADEPT_STATIC_MAX_LAYERS 64u
#define ADEPT_STATIC_MAX_BINS 256u
#define ADEPT_STATIC_MAX_MATERIALS 2u
int adept_step_static(const adept_geometry *geometry, const adept_tables *tables,
                      const adept_track *const tracks_in[3], const uint32_t n_in[3],
                      adept_track *const tracks_out[3], uint32_t out_capacity, uint32_t iterations,
                      void *cuda_stream, adept_result *out);
size_t adept_step_static_bytes(void);
const char *adept_step_static_error(void);

/* Elementary functions of the step, evaluated on the device for bit-equality tests against the
 * oracle (DESIGN.md rules R1, R3, M8-M10, T13).  in/out are DEVICE arrays; n = element count.
 *  fn 0: Philox-4x32-10; in = n x {ctr[4], key[2]} u32, out = n x 4 u32
 *  fn 1: u01;            in = n u32,  out = n f32
 *  fn 2: lg;             in = n f32,  out = n f32
 *  fn 3: ex;             in = n f32,  out = n f32
 *  fn 4: sincos2pi;      in = n f32,  out = n x {sin, cos} f32
 *  fn 5: in-range division (rule M11, csrc/mathfn.cuh); in = n x {a, b} f32, out = n f32 = a / b */
int adept_dev_math(int fn, const void *in, void *out, uint64_t n, void *cuda_stream);

#ifdef __cplusplus
}
#endif
#endif /* ADEPT_B200_H */
