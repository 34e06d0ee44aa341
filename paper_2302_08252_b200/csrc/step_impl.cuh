// The transport-step kernel and its helper kernels, templated on <layout, scheme, instrumented, CTA
// size (256 threads for small populations, 1024 for large ones: device_state.cuh)>.
//
// One launch = one iteration of all three per-type track buffers ("the tracks of each
// particle type are processed by a dedicated kernel"; here the three passes share one persistent
// grid so that an iteration costs one launch, and a tile always holds one type, so divergence
// between types never occurs inside a warp).  SURVEY.md §8(a) rows:
//   A0/A11  iteration control: counts live on the device, three deep by launch index; the first warp
//           of CTA 0 closes the previous launch and opens this one at kernel start (roll_iterations)
//           -- no host round trip, and no CTA that has to be the last;
//   A1      track load through the layout accessor (layout.cuh); dense scheme: the next tile is
//           fetched into shared memory by TMA while the current one is stepped;
//   A2-A8   the physics/geometry step (physics.cuh), tables staged in shared memory by one TMA
//           bulk copy per CTA and particle group.
//           The step is split (physics.cuh): every track takes the "move" half; tracks whose step ends
//           in a discrete interaction are parked in a shared-memory queue and the "interact" half
//           runs on dense batches of parked tracks, so that the Philox blocks and the sampling
//           code of rule S26 are executed by full warps instead of a few lanes per warp (the paper's
//           "diverging code paths");
//   A6      energy deposits go to per-CTA shared-memory bins in 64-bit fixed point (two native 32-bit
//           atomics; a 64-bit or fp64 shared-memory add would be a compare-and-swap loop);
//   A9      the warps of a group rank their outputs in arrival order with ONE shared-memory atomic
//           per warp on a packed word (3 x 9-bit counts + ticket); the last warp to arrive reserves
//           the group's output ranges with one global atomicAdd per destination type (dense: next
//           arrays; sparse: bump-allocated slots and the next slot lists);
//   A10     dense: survivors are written to the next array (whole record); sparse: only the words
//           that changed are written back in place, and the slot is pushed onto the next list;
//   A12     the instrumented instantiation counts every accessor call.
#pragma once
#include <cstdint>
#include <cstdlib>
#include <map>
#include <mutex>
#include <utility>
#include <cuda_runtime.h>

#include "device_state.cuh"
#include "layout.cuh"
#include "physics.cuh"

namespace adept {

// ---------------------------------------------------------------- small device utilities ------
// Barrier of one group of kGroup threads (named barrier 1 + group; barrier 0 is __syncthreads).
__device__ __forceinline__ void group_sync(int group) {
  asm volatile("bar.sync %0, %1;" ::"r"(group + 1), "n"(kGroup) : "memory");
}

// Variant bits of the step kernel (template parameter VAR): slot recycling of the sparse scheme
// (ADEPT_FLAG_RECYCLE_SLOTS) and the extended physics rules X36-X38 (adept_tables.physics = 1).
enum Variant : int { V_RECYCLE = 1, V_PHYS = 2, V_MSC = 4 };  // V_MSC (rule X39) comes with V_PHYS
__host__ __device__ constexpr int phys_of(int var) { return (var & V_MSC) ? 2 : ((var & V_PHYS) ? 1 : 0); }

// ---- section clocks (timing build only) ------------------------------------------------------------
// BASELINE.json configs[3]: "each scheme reports step plus slot-allocation/compaction time".  Allocation
// and compaction are fused into the step kernel (rows A9, A10), so a variant of the library compiled
// with -DADEPT_TIMING_SECTIONS brackets the sections of a tile with clock64(): lane 0 of every warp adds
// the cycles it spent in each section to CTA counters, flushed to Params::sections at kernel end.
// The shares of the per-warp cycles, applied to the kernel time of the normal build, are the reported
// per-section times.  In the normal build the clock is an empty object.
enum Section : int {
  SEC_OTHER = 0,     // launch prologue, table staging, loop control, tally flush
  SEC_LOAD = 1,      // A1: waiting for / fetching the records of a tile
  SEC_PHYSICS = 2,   // A2-A7: the move half and its scoring
  SEC_INTERACT = 3,  // A8: the interact half (queue read, sampling, scoring)
  SEC_ALLOC = 4,     // A9: ballots, arrival word, range / slot reservation, the group barrier, ranks
  SEC_STORE = 5,     // A10: survivor and secondary writes, slot-list pushes, parked-queue writes
  kNumSections = 8
};
#ifdef ADEPT_TIMING_SECTIONS
struct SectClock {
  long long t;
  uint32_t *acc;  // shared, [kNumSections]
  bool lead;
  __device__ __forceinline__ void start(uint32_t *a, bool l) { acc = a; lead = l; t = clock64(); }
  __device__ __forceinline__ void mark(int s) {
    const long long n = clock64();
    if (lead) atomicAdd(&acc[s], static_cast<uint32_t>(n - t));
    t = n;
  }
};
#else
struct SectClock {
  __device__ __forceinline__ void start(uint32_t *, bool) {}
  __device__ __forceinline__ void mark(int) {}
};
#endif

// ---- tally bins (row A6) -------------------------------------------------------------------------
struct Bins {
  uint32_t *lo, *hi;  // shared, n_slabs + 1 entries each
};
// bins[bin] += x, x >= 0 an fp32 term in MeV, in 64-bit fixed point of unit 2^-32 MeV (device_state.cuh).
__device__ __forceinline__ void bin_add(const Bins &b, uint32_t bin, float x) {
  const unsigned long long f = __float2ull_rn(x * 4294967296.0f);
  const uint32_t l = static_cast<uint32_t>(f), h = static_cast<uint32_t>(f >> 32);
  const uint32_t old = atomicAdd(&b.lo[bin], l);
  const uint32_t up = h + ((old + l < old) ? 1u : 0u);  // carry out of the low limb
  if (up) atomicAdd(&b.hi[bin], up);
}

// ---- asynchronous tile prefetch (dense scheme) ---------------------------------------------------
// A tile of kGroup consecutive slots is contiguous in global memory per layout (AoS: one run of
// 64-byte records; AoSoA-32: 1792-byte blocks back to back; SoA: one run per field), so the next
// tile is fetched into shared memory by TMA bulk copies while the current one is being stepped:
// the global load latency leaves the critical path and no load instruction or address arithmetic
// is issued.
__device__ __forceinline__ void mbar_init(uint64_t *mbar, uint32_t count) {
  asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(static_cast<uint32_t>(__cvta_generic_to_shared(mbar))),
               "r"(count));
}
__device__ __forceinline__ void mbar_wait(uint64_t *mbar, uint32_t parity) {
  const uint32_t bar = static_cast<uint32_t>(__cvta_generic_to_shared(mbar));
  uint32_t done = 0;
  while (!done) {
    asm volatile(
        "{\n .reg .pred p;\n mbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n selp.u32 %0, 1, 0, p;\n}"
        : "=r"(done)
        : "r"(bar), "r"(parity)
        : "memory");
  }
}
__device__ __forceinline__ void bulk_g2s(void *smem_dst, const void *gmem_src, uint32_t bytes, uint64_t *mbar) {
  asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];" ::"r"(
                   static_cast<uint32_t>(__cvta_generic_to_shared(smem_dst))),
               "l"(gmem_src), "r"(bytes), "r"(static_cast<uint32_t>(__cvta_generic_to_shared(mbar)))
               : "memory");
}
// shared-memory counter += 1 with release/acquire ordering at CTA scope; returns the old value
__device__ __forceinline__ uint32_t arrive_acq_rel(uint32_t *counter) {
  uint32_t old;
  asm volatile("atom.acq_rel.cta.shared::cta.add.u32 %0, [%1], 1;"
               : "=r"(old)
               : "r"(static_cast<uint32_t>(__cvta_generic_to_shared(counter)))
               : "memory");
  return old;
}

// Called by ONE thread, after every warp of the group has taken its records out of `in_buf`.
template <int L>
__device__ __forceinline__ void prefetch_tile(const Params &p, int kind, uint32_t par, uint32_t tile, uint32_t n_kind,
                                              uint32_t *in_buf, uint64_t *mbar) {
  const uint32_t *rec = p.kind[kind].rec[par];
  const uint32_t first = tile * kGroup;
  const uint32_t n = (n_kind - first < uint32_t(kGroup)) ? n_kind - first : uint32_t(kGroup);
  asm volatile("fence.proxy.async.shared::cta;" ::: "memory");  // generic reads of in_buf before async writes
  const uint32_t bar = static_cast<uint32_t>(__cvta_generic_to_shared(mbar));
  if constexpr (L == L_SOA) {
    // The SoA buffer is a 2-D tensor [14 fields][capacity slots]; a tile is the box [14][kGroup] of
    // it: ONE tiled TMA copy through the tensor map of this kind's buffer (encoded at adept_create),
    // landing field-major in shared memory -- the SoA mapping with capacity kGroup.  Slots are padded
    // to whole tiles, so the box of a ragged last tile stays inside the tensor.
    (void)rec; (void)n;
    constexpr uint32_t bytes = uint32_t(kGroup) * kNumFields * 4u;
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(bar), "r"(bytes) : "memory");
    asm volatile(
        "cp.async.bulk.tensor.2d.shared::cluster.global.tile.mbarrier::complete_tx::bytes [%0], [%1, {%2, %3}], [%4];" ::"r"(
            static_cast<uint32_t>(__cvta_generic_to_shared(in_buf))),
        "l"(reinterpret_cast<uint64_t>(&p.tile_map[kind][par])), "r"(first), "r"(0u), "r"(bar)
        : "memory");
  } else if constexpr (L == L_AOS) {
    // The AoS buffer is a 2-D tensor [capacity][16 words]; a tile is the box [kGroup][16], copied
    // with the 64-byte swizzle: the 16-byte chunk c of row r lands at chunk c ^ ((address >> 7) & 3),
    // so that the threads of a quarter warp, which each read one chunk of their own 64-byte record,
    // hit different banks (a linear copy makes those loads 4-way bank conflicts).
    (void)rec; (void)n;
    constexpr uint32_t bytes = uint32_t(kGroup) * 64u;
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(bar), "r"(bytes) : "memory");
    asm volatile(
        "cp.async.bulk.tensor.2d.shared::cluster.global.tile.mbarrier::complete_tx::bytes [%0], [%1, {%2, %3}], [%4];" ::"r"(
            static_cast<uint32_t>(__cvta_generic_to_shared(in_buf))),
        "l"(reinterpret_cast<uint64_t>(&p.tile_map[kind][par])), "r"(0u), "r"(first), "r"(bar)
        : "memory");
  } else if constexpr (L == L_SOA16 || L == L_HC16) {  // four runs: three of 16-byte vectors, one of 8-byte vectors
    const uint32_t n2 = (n + 1u) & ~1u;  // whole 16-byte pieces (slots are padded to whole tiles)
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(bar), "r"(n2 * 56u) : "memory");
#pragma unroll
    for (int gI = 0; gI < 4; ++gI)
      bulk_g2s(in_buf + Mapping<L_SOA16>::index(kGroup, 0, 4 * gI), rec + Mapping<L_SOA16>::index(p.capacity, first, 4 * gI),
               n2 * (gI < 3 ? 16u : 8u), mbar);
  } else {  // AoSoA-n: whole blocks, one contiguous run
    constexpr uint32_t kL = Mapping<L>::kLanes;
    static_assert(kL <= uint32_t(kGroup), "a staged tile holds whole AoSoA blocks");
    const uint32_t bytes = ((n + kL - 1u) / kL) * (kL * kNumFields * 4u);
    const uint32_t *src = rec + size_t(first / kL) * (kL * kNumFields);
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(bar), "r"(bytes) : "memory");
    bulk_g2s(in_buf, src, bytes, mbar);
  }
}

// The thread's record out of the staged tile (same mapping as in global memory, capacity = kGroup).
template <int L> __device__ __forceinline__ Trk staged_load(const uint32_t *in_buf, int gtid, int kind = 2) {
  Trk t;
  if constexpr (L == L_HC16) {
    using V = Mapping<L_SOA16>;
    const uint4 a = *reinterpret_cast<const uint4 *>(in_buf + V::index(kGroup, gtid, 0));
    const uint4 b = *reinterpret_cast<const uint4 *>(in_buf + V::index(kGroup, gtid, 4));
    const uint4 c = *reinterpret_cast<const uint4 *>(in_buf + V::index(kGroup, gtid, 8));
    const uint2 d = *reinterpret_cast<const uint2 *>(in_buf + V::index(kGroup, gtid, 12));
    return hc16_unpack(kind == 2, a, b, c, d);
  }
  if constexpr (L == L_AOS) {
    // undo the copy's 64-byte swizzle (prefetch_tile): chunk c of this thread's record is at chunk
    // c ^ s of its row, s = bits 7-8 of the row's shared-memory address
    const uint32_t row = static_cast<uint32_t>(__cvta_generic_to_shared(in_buf)) + uint32_t(gtid) * 64u;
    const uint32_t sw = ((row >> 7) & 3u) << 4;
    uint4 a, b, c;
    uint2 d;
    asm volatile("ld.shared.v4.u32 {%0, %1, %2, %3}, [%4];" : "=r"(a.x), "=r"(a.y), "=r"(a.z), "=r"(a.w) : "r"(row + (0u ^ sw)));
    asm volatile("ld.shared.v4.u32 {%0, %1, %2, %3}, [%4];" : "=r"(b.x), "=r"(b.y), "=r"(b.z), "=r"(b.w) : "r"(row + (16u ^ sw)));
    asm volatile("ld.shared.v4.u32 {%0, %1, %2, %3}, [%4];" : "=r"(c.x), "=r"(c.y), "=r"(c.z), "=r"(c.w) : "r"(row + (32u ^ sw)));
    asm volatile("ld.shared.v2.u32 {%0, %1}, [%2];" : "=r"(d.x), "=r"(d.y) : "r"(row + (48u ^ sw)));
    t.px = __uint_as_float(a.x); t.py = __uint_as_float(a.y); t.pz = __uint_as_float(a.z);
    t.dx = __uint_as_float(a.w); t.dy = __uint_as_float(b.x); t.dz = __uint_as_float(b.y);
    t.ekin = __uint_as_float(b.z); t.n0 = __uint_as_float(b.w);
    t.n1 = __uint_as_float(c.x); t.n2 = __uint_as_float(c.y);
    t.vol = c.z; t.id_lo = c.w; t.id_hi = d.x; t.step = d.y;
  } else if constexpr (L == L_SOA16) {
    const uint4 a = *reinterpret_cast<const uint4 *>(in_buf + Mapping<L>::index(kGroup, gtid, 0));
    const uint4 b = *reinterpret_cast<const uint4 *>(in_buf + Mapping<L>::index(kGroup, gtid, 4));
    const uint4 c = *reinterpret_cast<const uint4 *>(in_buf + Mapping<L>::index(kGroup, gtid, 8));
    const uint2 d = *reinterpret_cast<const uint2 *>(in_buf + Mapping<L>::index(kGroup, gtid, 12));
    t.px = __uint_as_float(a.x); t.py = __uint_as_float(a.y); t.pz = __uint_as_float(a.z);
    t.dx = __uint_as_float(a.w); t.dy = __uint_as_float(b.x); t.dz = __uint_as_float(b.y);
    t.ekin = __uint_as_float(b.z); t.n0 = __uint_as_float(b.w);
    t.n1 = __uint_as_float(c.x); t.n2 = __uint_as_float(c.y);
    t.vol = c.z; t.id_lo = c.w; t.id_hi = d.x; t.step = d.y;
  } else {
#pragma unroll
    for (int f = 0; f < kNumFields; ++f) trk_set_word(t, f, in_buf[Mapping<L>::index(kGroup, gtid, f)]);
  }
  return t;
}

// ---- asynchronous record gather (sparse scheme) --------------------------------------------------
// The slot list is dense, the records it names are not.  One tile ahead of the tile being stepped,
// every thread copies the record of ITS next list entry into the group's staging buffer with cp.async,
// and its list entry for the tile after that into a stash word -- no register holds a value that is
// still in flight, so nothing waits for a load until the tile is reached (cp.async.wait_group).
//   AoS: four lanes fetch one 64-byte record (lane l: piece l & 3 of the record of lane 8 j + (l >> 2),
//        j = 0..3), so that a warp's copy asks for 8 whole records = whole sectors; the pieces land
//        record-major with the 64-byte swizzle of the dense tiles (staged_load<L_AOS> undoes it).
//   The other layouts load their records directly (Mapping<L>::kSparseGather = false): for SoA / AoSoA-n
//        a record is 14 scattered words -- the sector amplification the paper reports (PAPER.md:111,
//        145) -- and 14 four-byte copies plus the L1 capacity given up for the staging buffer cost more
//        than the latency they hide; SoA16 gains only above ~80 % occupancy.
constexpr uint32_t kNoSlot = 0xFFFFFFFFu;
__device__ __forceinline__ void cp_async_16(uint32_t smem_dst, const void *gmem_src) {  // .cg: not kept in L1
  asm volatile("cp.async.cg.shared.global [%0], [%1], 16;" ::"r"(smem_dst), "l"(gmem_src) : "memory");
}
__device__ __forceinline__ void cp_async_4(uint32_t smem_dst, const void *gmem_src) {
  asm volatile("cp.async.ca.shared.global [%0], [%1], 4;" ::"r"(smem_dst), "l"(gmem_src) : "memory");
}
__device__ __forceinline__ void cp_async_commit() { asm volatile("cp.async.commit_group;" ::: "memory"); }
__device__ __forceinline__ void cp_async_wait_all() { asm volatile("cp.async.wait_group 0;" ::: "memory"); }

// `slot` = kNoSlot for a thread without a list entry (ragged last tile).  Called by whole warps.
template <int L>
__device__ __forceinline__ void gather_record(const uint32_t *rec, uint32_t cap, uint32_t slot, uint32_t *in_buf, int gtid) {
  const uint32_t row = static_cast<uint32_t>(__cvta_generic_to_shared(in_buf));
  if constexpr (L == L_AOS) {
    const int lane = gtid & 31, piece = lane & 3;
    const uint32_t warp_row = uint32_t(gtid & ~31);
#pragma unroll
    for (int j = 0; j < 4; ++j) {
      const int src = 8 * j + (lane >> 2);
      const uint32_t s_src = __shfl_sync(0xFFFFFFFFu, slot, src);
      const uint32_t dst_row = row + (warp_row + uint32_t(src)) * 64u;
      const uint32_t sw = ((dst_row >> 7) & 3u) << 4;
      if (s_src != kNoSlot)
        cp_async_16(dst_row + ((uint32_t(piece) << 4) ^ sw), rec + size_t(s_src) * Mapping<L>::kStride + piece * 4);
    }
  } else {  // generic form (no layout uses it today: the word-by-word layouts load directly)
    if (slot != kNoSlot) {
#pragma unroll
      for (int f = 0; f < kNumFields; ++f)
        cp_async_4(row + uint32_t(f * kGroup + gtid) * 4u, rec + Mapping<L>::index(cap, slot, f));
    }
  }
}
// The thread's gathered record out of the staging buffer.
template <int L> __device__ __forceinline__ Trk gathered_load(const uint32_t *in_buf, int gtid) {
  if constexpr (L == L_AOS) return staged_load<L>(in_buf, gtid);
  Trk t;
#pragma unroll
  for (int f = 0; f < kNumFields; ++f) trk_set_word(t, f, in_buf[f * kGroup + gtid]);
  return t;
}
// Issue the gather of the record in `slot` (this thread's entry of tile `tile_next`), remember the slot,
// and fetch the thread's list entry of the tile after that into the stash.  stash = in_buf + tile words:
// [0][gtid] slot of the gathered record, [1][gtid] list entry of the following tile.
template <int L>
__device__ __forceinline__ void gather_ahead(const Params &p, int kind, uint32_t par, uint32_t slot, uint32_t i_after,
                                             uint32_t n_kind, uint32_t *in_buf, int gtid) {
  uint32_t *stash = in_buf + Mapping<L>::words(kGroup);
  gather_record<L>(p.kind[kind].rec[0], p.capacity, slot, in_buf, gtid);
  stash[gtid] = slot;
  if (i_after < n_kind)
    cp_async_4(static_cast<uint32_t>(__cvta_generic_to_shared(stash + kGroup + gtid)), p.kind[kind].queue[par] + i_after);
  else
    stash[kGroup + gtid] = kNoSlot;
  cp_async_commit();
}

template <int L, bool INSTR>
__device__ __forceinline__ TrackView<L, INSTR> make_view(const Params &p, int kind, int buf, uint32_t *cta_probe) {
  TrackView<L, INSTR> v;
  v.base = p.kind[kind].rec[buf];
  v.cap = p.capacity;
  v.storage_off = size_t(buf) * Mapping<L>::words(p.capacity) * 4;
  v.buf_index = uint32_t(buf);
  v.kind = kind;
  v.sink.cta_field_rw = cta_probe + kind * (kNumFields * 2);
  v.sink.lines = p.kind[kind].instr_lines;
  v.sink.slots = p.kind[kind].instr_slots;
  return v;
}

__device__ __forceinline__ Trk kid_track(const Trk &parent, const Kid &k) {
  Trk c;
  c.px = parent.px; c.py = parent.py; c.pz = parent.pz;
  c.dx = k.dx; c.dy = k.dy; c.dz = k.dz;
  c.ekin = k.ekin;
  c.n0 = -1.0f; c.n1 = -1.0f; c.n2 = -1.0f;
  c.vol = parent.vol;
  c.id_lo = k.id_lo; c.id_hi = k.id_hi;
  c.step = 0u;
  return c;
}

// ---- rule X39: the side array of the three multiple-scattering words (e- and e+ only) --------------
__device__ __forceinline__ void msc_store(const Params &p, int kind, int buf, uint32_t idx, float m0, float m1, float m2) {
  float *a = p.kind[kind].msc[buf];
  a[idx] = m0;
  a[size_t(p.capacity) + idx] = m1;
  a[2 * size_t(p.capacity) + idx] = m2;
}
__device__ __forceinline__ void msc_load(const Params &p, int kind, int buf, uint32_t idx, Trk &t) {
  const float *a = p.kind[kind].msc[buf];
  t.m0 = a[idx];
  t.m1 = a[size_t(p.capacity) + idx];
  t.m2 = a[2 * size_t(p.capacity) + idx];
}

// ---- parked tracks (the queue between the two halves of the step) ----------------------------------
// Entry q = 7 (sparse: 8) 64-bit words; the pending interaction rides in the top bits of the step word.
// (dense scheme with multiple scattering: two more 64-bit words carry the track's three cold words)
template <int SCHEME, bool MSC = false>
__device__ __forceinline__ void park_store(uint32_t *queue, uint32_t q, const Trk &t, int pending, uint32_t slot) {
  uint2 *e = reinterpret_cast<uint2 *>(queue + size_t(q) * queue_words(SCHEME, MSC));
  if (SCHEME == S_DENSE && MSC) {
    e[7] = make_uint2(__float_as_uint(t.m0), __float_as_uint(t.m1));
    e[8] = make_uint2(__float_as_uint(t.m2), 0u);
  }
#pragma unroll
  for (int f = 0; f < 12; f += 2) e[f / 2] = make_uint2(trk_word(t, f), trk_word(t, f + 1));
  e[6] = make_uint2(t.id_hi, t.step | (uint32_t(pending) << 29));
  if (SCHEME == S_SPARSE) e[7] = make_uint2(slot, 0u);
}
template <int SCHEME, bool MSC = false>
__device__ __forceinline__ void park_load(const uint32_t *queue, uint32_t q, Trk &t, int &pending, uint32_t &slot) {
  const uint2 *e = reinterpret_cast<const uint2 *>(queue + size_t(q) * queue_words(SCHEME, MSC));
  if (SCHEME == S_DENSE && MSC) {
    const uint2 a = e[7], b = e[8];
    t.m0 = __uint_as_float(a.x); t.m1 = __uint_as_float(a.y); t.m2 = __uint_as_float(b.x);
  }
#pragma unroll
  for (int f = 0; f < 12; f += 2) {
    const uint2 w = e[f / 2];
    trk_set_word(t, f, w.x);
    trk_set_word(t, f + 1, w.y);
  }
  const uint2 w = e[6];
  t.id_hi = w.x;
  t.step = w.y & 0x1FFFFFFFu;
  pending = int(w.y >> 29);
  if (SCHEME == S_SPARSE) slot = e[7].x;
}

// ---- arrival word (row A9) -----------------------------------------------------------------------
// Three 9-bit counts (bits 0-8, 9-17, 18-26) and a ticket (bits 27-29).  Every warp of a group adds
// its counts and one ticket with a single shared-memory atomic; what the atomic returns are the
// counts of the warps that arrived before it = the warp's ranks.  The warp that draws the last ticket
// knows the group's totals.
constexpr uint32_t kCountMask = 511u;
constexpr uint32_t kTicket = 1u << 27;
__device__ __forceinline__ uint32_t count_of(uint32_t word, int field) { return (word >> (9 * field)) & kCountMask; }
__device__ __forceinline__ bool last_ticket(uint32_t old) { return (old >> 27) == uint32_t(kWarpsPerGroup - 1); }

// Per-group shared state.
struct GroupShared {
  uint64_t mbar_in;      // completion of the staged tile
  uint32_t loaded;       // warps that have taken their records out of the staged tile (monotonic)
  uint32_t acc[2];       // arrival words, alternating between consecutive tiles / batches
  uint32_t qtot[2];      // parked tracks after the tile
  uint32_t base[2][4];   // first output entry per destination kind (dense: next array; sparse: next slot list)
  uint32_t sbase[2][4];  // sparse: first new (bump-allocated) slot per destination kind
  // sparse scheme with slot recycling: tracks that end in each warp of the tile / batch, where the
  // group's freed slots go in the ring, and per destination kind the ring position and number of
  // recycled slots its children take before bump-allocated ones
  uint32_t kcnt[2][kWarpsPerGroup];
  uint32_t fbase[2];
  uint32_t rbase[2][4], rn[2][4];
  uint32_t sgot[2][4];   // sparse: children per destination kind that got a slot (the rest are dropped: overflow)
};
// Per-CTA shared state.
struct CtaShared {
  uint64_t mbar;  // completion of the staged tables
  uint32_t alive[4];
  uint32_t escaped[4];
  uint32_t probe[3 * kNumFields * 2];
  uint32_t sect[kNumSections];  // timing build: cycles per section (lane 0 of every warp)
  GroupShared grp[kMaxGroupsPerCta];
};

// A11 / A0 (see Ctl, device_state.cuh).  Run by one warp, lane k < 3 = kind k, so that the dependent
// global accesses of the three kinds overlap: the first warp of CTA 0 at the start of launch `it`
// (open = true), and close_kernel before the host reads the control block (open = false).
// close: every launch below `it` that is still open gets its statistics added to the cumulative
// counters and its buffers cleared for the launch two after it.  open: launch `it` is counted.
template <bool SPARSE, bool RECYCLE>
__device__ __forceinline__ void roll_iterations(Ctl *c, uint32_t capacity, uint32_t it, bool open, int lane
#ifdef ADEPT_TIMING_SECTIONS
                                                , unsigned long long *sections
#endif
) {
  const int k = lane < 3 ? lane : 0;
  // normally one launch (it - 1) is open, or none; more than two can only mean that the launch index was
  // set without the workspace copy that belongs to it (adept.h "Workspace"): then nothing is closed
  uint32_t first = c->closed;
  if ((it >= first ? it - first : it + (kLaunchWrap - first)) > 2u) first = it;
  for (uint32_t j = first; j != it; j = next_launch(j)) {
    const uint32_t b = j % 3u, b1 = (j + 1u) % 3u;
    if (lane < 3) {
      const uint32_t raw = c->n[b][k], n = raw < capacity ? raw : capacity;
      const uint32_t out = __ldcg(&c->n[b1][k]);
      const uint32_t alive = __ldcg(&c->alive[b][k]), esc = __ldcg(&c->esc[b][k]);
      const unsigned long long killed = c->killed[k], escaped = c->escaped_n[k], secondaries = c->secondaries[k],
                               used = c->slots_used[k];
      c->killed[k] = killed + (n - alive);
      c->escaped_n[k] = escaped + esc;
      c->secondaries[k] = secondaries + (out - alive);
      if (out > capacity) c->overflow = 1u;
      if (SPARSE) {
        uint32_t top = __ldcg(&c->slot_top[k]);
        // after an overflow the clamped top is written back: the host may enqueue up to a burst of further
        // launches before it sees the flag, and an allocator that kept counting could wrap past 2^32 and
        // hand out live slots again
        if (top > capacity) { top = capacity; c->overflow = 1u; c->slot_top[k] = capacity; }
        if (top > used) c->slots_used[k] = top;
      } else {
        const uint32_t live = out < capacity ? out : capacity;
        if (live > used) c->slots_used[k] = live;
      }
      c->n[b][k] = 0u; c->alive[b][k] = 0u; c->esc[b][k] = 0u;
      if (SPARSE && RECYCLE) c->ring_tail[b][k] = 0u;
    }
#ifdef ADEPT_TIMING_SECTIONS
    if (lane == 0) {  // launch timeline: first CTA start -> last CTA end of launch j (ns)
      unsigned long long *w = sections + kNumSections + 2u * (j & 1u);  // scratch of launch j: {min start, max end}
      if (w[1] > w[0] && w[0] != ~0ull) sections[6] += w[1] - w[0];
      w[0] = ~0ull;
      w[1] = 0ull;
    }
#endif
  }
  __syncwarp();
  const uint32_t bi = it % 3u;
  uint32_t n_now = 0u;
  if (lane < 3) {
    const uint32_t raw = c->n[bi][k];
    n_now = raw < capacity ? raw : capacity;
  }
  const uint32_t live = __reduce_add_sync(0xFFFFFFFFu, n_now);
  if (lane < 3) {
    if (SPARSE && live == 0u) {  // rule S30: slots are reused (without recycling: only) once the buffer is empty
      c->slot_top[k] = 0u; c->free_head[k] = 0u; c->free_tail[k] = 0u;
      c->ring_tail[0][k] = 0u; c->ring_tail[1][k] = 0u; c->ring_tail[2][k] = 0u;
    }
    if (open) {
      c->steps[k] += n_now;
      // the tail of the free ring at the start of launch it + 1 = the tail at the start of this launch
      // + what this launch pushes (added by the pushing groups themselves)
      if (SPARSE && RECYCLE && live != 0u) atomicAdd(&c->ring_tail[(it + 1u) % 3u][k], c->ring_tail[bi][k]);
    } else {
      c->n_cur[k] = n_now;  // summary for the host
    }
  }
  if (lane == 0) {
    c->closed = it;
    if (open) { if (live) c->iterations += 1ull; }
    else c->parity = it & 1u;
  }
}

// ------------------------------------------------------------------- tile = kGroup tracks -----
template <int KIND> __device__ __forceinline__ constexpr int kid_kind(int ordinal) {
  return KIND == K_GAMMA ? (ordinal == 0 ? K_EM : K_EP) : K_GAMMA;  // rule R5
}

// What a group carries through its tiles.
struct GroupRefs {
  CtaShared *cta;
  GroupShared *g;
  Bins bins;         // shared, CTA-wide
  uint32_t *queue;   // shared, [kQueueCap][queue_words]
  uint32_t *in_buf;  // shared, one staged tile (dense scheme)
  int group, gtid;   // group index inside the CTA, thread index inside the group
  SectClock *clk;    // timing build: this thread's section clock
};

// S25 / S31 energy of a track that leaves the simulation
template <int KIND> __device__ __forceinline__ void bin_add_track_energy(const Bins &b, uint32_t bin, float ekin) {
  bin_add(b, bin, ekin);
  if (KIND == K_EP) bin_add(b, bin, two_mc2());
}

// First half of the step for tile `tile` of kind KIND's current set (rows A1-A7, A10 for the
// tracks whose step ends without an interaction).  `queued` = parked tracks of the group before
// the tile; returns the number after it (the same value in every thread of the group).
template <int L, int SCHEME, bool INSTR, int VAR, int KIND>
__device__ __forceinline__ uint32_t move_tile(const Params &p, const Env &env, const GroupRefs &c, uint32_t par,
                                              uint32_t tile, uint32_t next_tile, uint32_t n_kind, int sbuf,
                                              uint32_t &in_phase, uint32_t queued, bool l2_prefetch) {
  const int gtid = c.gtid, lane = gtid & 31;
  const uint32_t lt_mask = (1u << lane) - 1u;
  const uint32_t i = tile * kGroup + gtid;
  const bool active = i < n_kind;
  Ctl *ctl = p.ctl;
  GroupShared &g = *c.g;

  // A1: load
  c.clk->mark(SEC_OTHER);
  uint32_t slot = i;
  constexpr bool kGather = SCHEME == S_SPARSE && Mapping<L>::kSparseGather;

  const TrackView<L, INSTR> cur = make_view<L, INSTR>(p, KIND, (SCHEME == S_DENSE) ? int(par) : 0, c.cta->probe);
  Trk t, old;
  uint32_t vol_before = 0u;
  MoveOut o;
  move_out_init(o);
  o.alive = false;
  if (SCHEME == S_DENSE) {  // the tile was staged in shared memory by prefetch_tile
    mbar_wait(&g.mbar_in, in_phase);
    in_phase ^= 1u;
    if (active) t = staged_load<L>(c.in_buf, gtid, KIND);
    // the warp has its records in registers; the last warp to get there refills the staging buffer
    // with the group's next tile, which then loads while this one is stepped
    __syncwarp();
    if (lane == 0) {
      const uint32_t arrived = arrive_acq_rel(&g.loaded);
      if ((arrived % uint32_t(kWarpsPerGroup)) == uint32_t(kWarpsPerGroup - 1) && next_tile != 0xFFFFFFFFu)
        prefetch_tile<L>(p, KIND, par, next_tile, n_kind, c.in_buf, &g.mbar_in);
    }
  }
  if constexpr (kGather) {  // the record was gathered into the staging buffer one tile ago (gather_ahead)
    uint32_t *stash = c.in_buf + Mapping<L>::words(kGroup);
    cp_async_wait_all();
    if (L == L_AOS) __syncwarp();  // the pieces of a record were copied by four lanes of the warp
    slot = stash[gtid];
    const uint32_t s_next = stash[kGroup + gtid];
    if (active) t = gathered_load<L>(c.in_buf, gtid);
    if (next_tile != 0xFFFFFFFFu) {
      if (L == L_AOS) __syncwarp();  // every lane has read its record: the rows may be refilled
      const uint32_t i_after = (2u * next_tile - tile) * kGroup + gtid;  // next_tile - tile = groups of the grid
      gather_ahead<L>(p, KIND, par, s_next, i_after, n_kind, c.in_buf, gtid);
    }
  } else if (SCHEME == S_SPARSE) {
    // Word-by-word layouts: plain loads of the record the list entry names.  The list entries
    // themselves run two tiles ahead (cp.async into two stash words per thread, roles alternating by
    // tile), so the record loads do not wait for them, and the lines of the next tile's record are
    // requested into L2 while this tile is stepped.
    uint32_t *stash = c.in_buf;
    cp_async_wait_all();
    slot = stash[in_phase * kGroup + gtid];
    const uint32_t s_next = stash[(in_phase ^ 1u) * kGroup + gtid];
    if (next_tile != 0xFFFFFFFFu) {
      const uint32_t i_after = (2u * next_tile - tile) * kGroup + gtid;  // the group's tile after next
      if (i_after < n_kind)
        cp_async_4(static_cast<uint32_t>(__cvta_generic_to_shared(stash + in_phase * kGroup + gtid)), p.kind[KIND].queue[par] + i_after);
      else
        stash[in_phase * kGroup + gtid] = kNoSlot;
      cp_async_commit();
      // worth it only where the slots in use are mostly live (measured: -3.5 % at 70-90 % occupancy,
      // +25 % at 10 %, where every prefetch is a sector of its own)
      if (l2_prefetch && s_next != kNoSlot) {
#pragma unroll
        for (int f = 0; f < kNumFields; ++f)
          if (L != L_SOA16 && L != L_HC16) {
            asm volatile("prefetch.global.L2 [%0];" ::"l"(p.kind[KIND].rec[0] + Mapping<L>::index(p.capacity, s_next, f)));
          } else if (f % 4 == 0) {  // one request per 16-byte vector
            asm volatile("prefetch.global.L2 [%0];" ::"l"(p.kind[KIND].rec[0] + Mapping<L_SOA16>::index(p.capacity, s_next, f)));
          }
      }
    }
    in_phase ^= 1u;
    if (active) t = cur.load(slot);
  }
  constexpr bool kMsc = (VAR & V_MSC) != 0 && KIND != K_GAMMA;
  if (kMsc && active) msc_load(p, KIND, (SCHEME == S_DENSE) ? int(par) : 0, slot, t);
  if (active) {
    if (INSTR && (SCHEME == S_DENSE || kGather)) {
#pragma unroll
      for (int f = 0; f < kNumFields; ++f) cur.probe(f, 0, slot);
    }
    if (INSTR && SCHEME == S_SPARSE) old = t;  // the counting build compares against the pre-step record
    vol_before = t.vol;
    c.clk->mark(SEC_LOAD);
    if constexpr (KIND == K_GAMMA) move_gamma(t, env, o);
    else move_elec<KIND, phys_of(VAR)>(t, env, o);
    // A6: scoring into the CTA's bins (pre-step slab; the S31 guard uses the post-step slab).  A
    // photon deposits nothing in this half; the rare terms share one branch.
    if (KIND != K_GAMMA && o.dep != 0.0f) bin_add(c.bins, vol_before, o.dep);
    if ((KIND != K_GAMMA && o.dep_b != 0.0f) || o.escaped || o.guard) {
      if (KIND != K_GAMMA && o.dep_b != 0.0f) bin_add(c.bins, vol_before, o.dep_b);
      if (o.escaped) bin_add_track_energy<KIND>(c.bins, env.n_slabs, t.ekin);
      if (o.guard) bin_add_track_energy<KIND>(c.bins, t.vol, t.ekin);
    }
  }
  c.clk->mark(SEC_PHYSICS);
  const bool parked = active && o.pending != P_NONE;
  const bool survives = active && !parked && o.alive;
  // A10 sparse: in-place update of the words that changed (parked tracks too: the interaction later
  // writes only what it changes).  Done first: it needs no rank, and the pre-step copy of the record
  // dies here instead of living through the ranking.
  if (SCHEME == S_SPARSE) {
    if (survives || parked) {
      if constexpr (INSTR) cur.store_changed(slot, t, old);  // counts exactly the words that changed
      else cur.template store_moved<KIND == K_GAMMA, (VAR & V_PHYS) != 0, (VAR & V_PHYS) != 0 && KIND == K_EP, kMsc>(slot, t, t.vol != vol_before);
      if (kMsc) msc_store(p, KIND, 0, slot, t.m0, t.m1, t.m2);
    }
    c.clk->mark(SEC_STORE);
  }
  const uint32_t m_surv = __ballot_sync(0xFFFFFFFFu, survives);
  const uint32_t m_esc = __ballot_sync(0xFFFFFFFFu, o.escaped);
  const uint32_t m_park = __ballot_sync(0xFFFFFFFFu, parked);
  // sparse scheme with slot recycling: a track that ends here frees its slot
  constexpr bool recycle = SCHEME == S_SPARSE && (VAR & V_RECYCLE) != 0;
  const bool ends = recycle && active && !parked && !survives;
  uint32_t m_end = 0u;
  if (SCHEME == S_SPARSE && recycle) {
    m_end = __ballot_sync(0xFFFFFFFFu, ends);
    if (lane == 0) g.kcnt[sbuf][gtid >> 5] = uint32_t(__popc(m_end));
  }

  // A9: rank survivors and parked tracks of the warp inside the group (the third count, escapes, is
  // only totalled); last warp reserves the range and books the tile's counts
  uint32_t word = 0;
  if (lane == 0) {
    const uint32_t mine = uint32_t(__popc(m_surv)) | (uint32_t(__popc(m_park)) << 9) | (uint32_t(__popc(m_esc)) << 18) | kTicket;
    word = atomicAdd(&g.acc[sbuf], mine);
    if (last_ticket(word)) {
      const uint32_t total = word + mine;
      g.acc[sbuf] = 0u;  // next used two tiles from now, behind a group barrier
      g.qtot[sbuf] = queued + count_of(total, 1);
      const uint32_t n_out = count_of(total, 0), n_esc = count_of(total, 2);
      g.base[sbuf][0] = n_out ? atomicAdd(&ctl->n[(p.it + 1u) % 3u][KIND], n_out) : 0u;
      if (n_out) atomicAdd(&c.cta->alive[KIND], n_out);
      if (n_esc) atomicAdd(&c.cta->escaped[KIND], n_esc);
      if (SCHEME == S_SPARSE && recycle) {
        const uint32_t first = tile * kGroup;
        const uint32_t n_tile = (n_kind - first < uint32_t(kGroup)) ? n_kind - first : uint32_t(kGroup);
        const uint32_t n_end = n_tile - n_out - count_of(total, 1);
        if (n_end) {
          g.fbase[sbuf] = atomicAdd(&ctl->free_tail[KIND], n_end);
          atomicAdd(&ctl->ring_tail[(p.it + 1u) % 3u][KIND], n_end);
        }
      }
    }
  }
  word = __shfl_sync(0xFFFFFFFFu, word, 0);

  c.clk->mark(SEC_ALLOC);
  // park the tracks that still owe an interaction
  if (parked) {
    const uint32_t q = queued + count_of(word, 1) + __popc(m_park & lt_mask);
    park_store<SCHEME, kMsc>(c.queue, q, t, o.pending, slot);
  }
  c.clk->mark(SEC_STORE);
  group_sync(c.group);
  c.clk->mark(SEC_ALLOC);
  if (survives) {
    const uint32_t dst = g.base[sbuf][0] + count_of(word, 0) + __popc(m_surv & lt_mask);
    if (dst < p.capacity) {
      if (SCHEME == S_DENSE) {
        make_view<L, INSTR>(p, KIND, int(par ^ 1u), c.cta->probe).store(dst, t);  // A10
        if (kMsc) msc_store(p, KIND, int(par ^ 1u), dst, t.m0, t.m1, t.m2);
      } else {
        p.kind[KIND].queue[par ^ 1u][dst] = slot;  // slot pushed onto the next list
      }
    } else {
      ctl->overflow = 1u;
    }
  }
  if (SCHEME == S_SPARSE && ends) {  // freed slot -> the kind's ring, in warp order inside the tile
    uint32_t r = uint32_t(__popc(m_end & lt_mask));
    for (int w = 0; w < (gtid >> 5); ++w) r += g.kcnt[sbuf][w];
    p.kind[KIND].free_ring[(g.fbase[sbuf] + r) % p.capacity] = slot;
  }
  c.clk->mark(SEC_STORE);
  return g.qtot[sbuf];
}

// Second half of the step on a dense batch of up to kGroup parked tracks taken from the top of the
// group's queue (rows A8, A9, A10).  Returns the number of tracks left in the queue.
template <int L, int SCHEME, bool INSTR, int VAR, int KIND>
__device__ __forceinline__ uint32_t interact_batch(const Params &p, const Env &env, const GroupRefs &c, uint32_t par,
                                                   uint32_t queued, int sbuf) {
  const int gtid = c.gtid, lane = gtid & 31;
  const uint32_t lt_mask = (1u << lane) - 1u;
  Ctl *ctl = p.ctl;
  GroupShared &g = *c.g;
  const uint32_t batch = queued < uint32_t(kGroup) ? queued : uint32_t(kGroup);
  const uint32_t first = queued - batch;

  c.clk->mark(SEC_OTHER);
  const bool have = uint32_t(gtid) < batch;
  Trk t, before_interaction;
  InteractOut o;
  interact_out_init(o);
  o.alive = false;
  uint32_t slot = 0;
  if (have) {
    const uint32_t q = first + gtid;
    int pending;
    park_load<SCHEME, (VAR & V_MSC) != 0 && KIND != K_GAMMA>(c.queue, q, t, pending, slot);
    before_interaction = t;
    if constexpr (KIND == K_GAMMA) interact_gamma<phys_of(VAR)>(t, pending, env, o);
    else interact_elec<KIND, phys_of(VAR)>(t, pending, env, o);
    if (o.dep != 0.0f) bin_add(c.bins, t.vol, o.dep);
    if (o.dep_b != 0.0f) bin_add(c.bins, t.vol, o.dep_b);
    if (o.guard) bin_add_track_energy<KIND>(c.bins, t.vol, t.ekin);
  }
  c.clk->mark(SEC_INTERACT);
  constexpr int Q0 = kid_kind<KIND>(0), Q1 = kid_kind<KIND>(1);  // never KIND itself
  const uint32_t m_alive = __ballot_sync(0xFFFFFFFFu, o.alive);
  constexpr bool recycle = SCHEME == S_SPARSE && (VAR & V_RECYCLE) != 0;
  const bool ends = recycle && have && !o.alive;  // the parent's slot is free from the next iteration on
  uint32_t m_end = 0u;
  if (SCHEME == S_SPARSE && recycle) {
    m_end = __ballot_sync(0xFFFFFFFFu, ends);
    if (lane == 0) g.kcnt[sbuf][gtid >> 5] = uint32_t(__popc(m_end));
  }
  // Extended physics (rule X36): child 0 of an e+- is a photon (bremsstrahlung) or an e- (delta ray).
  // Delta rays are ranked in a field of their own: field 0 = e- for e+ parents; for e- parents
  // field 1 (the e+ field, which an e- parent never uses), with destination kind e-.
  constexpr bool kDelta = (VAR & V_PHYS) != 0 && KIND != K_GAMMA;
  constexpr int FD = (KIND == K_EM) ? 1 : 0;
  const bool k0d = kDelta && o.kid[0].kind == K_EM;
  const uint32_t m_k0 = __ballot_sync(0xFFFFFFFFu, o.kid[0].kind >= 0 && !k0d);
  const uint32_t m_kd = kDelta ? __ballot_sync(0xFFFFFFFFu, k0d) : 0u;
  const uint32_t m_k1 = __ballot_sync(0xFFFFFFFFu, o.kid[1].kind >= 0);
  auto dest_of = [](int field) -> int { return (kDelta && field == FD) ? int(K_EM) : field; };

  // A9: one arrival per warp with its output counts per destination kind
  uint32_t word = 0;
  if (lane == 0) {
    const uint32_t mine = (uint32_t(__popc(m_alive)) << (9 * KIND)) + (uint32_t(__popc(m_k0)) << (9 * Q0)) +
                          (uint32_t(__popc(m_k1)) << (9 * Q1)) + (uint32_t(__popc(m_kd)) << (9 * FD)) + kTicket;
    word = atomicAdd(&g.acc[sbuf], mine);
    if (last_ticket(word)) {
      const uint32_t total = word + mine;
      g.acc[sbuf] = 0u;
      if (count_of(total, KIND)) atomicAdd(&c.cta->alive[KIND], count_of(total, KIND));  // parents that survive
#pragma unroll
      for (int q = 0; q < 3; ++q) {
        const uint32_t want = count_of(total, q);
        const int d = dest_of(q);  // destination kind of field q
        uint32_t got = want;
        if (SCHEME == S_SPARSE && q != KIND) {
          // sparse: children get bump-allocated, never recycled slots (rule S30) -- or, with slot
          // recycling, first the slots freed up to the previous iteration (the kind's ring below
          // free_tail_start), then bump-allocated ones
          uint32_t n_ring = 0u, h = 0u;
          if (recycle && want) {
            h = atomicAdd(&ctl->free_head[d], want);
            const int32_t avail = static_cast<int32_t>(ctl->ring_tail[p.it % 3u][d] - h);
            n_ring = avail <= 0 ? 0u : (uint32_t(avail) < want ? uint32_t(avail) : want);
            if (n_ring != want) atomicSub(&ctl->free_head[d], want - n_ring);  // the head never passes the allocatable tail
          }
          g.rbase[sbuf][q] = h;
          g.rn[sbuf][q] = n_ring;
          const uint32_t rest = want - n_ring;
          const uint32_t sb = rest ? atomicAdd(&ctl->slot_top[d], rest) : 0u;
          g.sbase[sbuf][q] = sb;
          // slots past the end of the buffer do not exist: those children are dropped (overflow), and
          // only children that have a slot get a list entry, so every list entry names a real slot
          const uint32_t usable = (sb >= p.capacity) ? 0u : ((p.capacity - sb < rest) ? p.capacity - sb : rest);
          got = n_ring + usable;
          g.sgot[sbuf][q] = got;
        }
        g.base[sbuf][q] = got ? atomicAdd(&ctl->n[(p.it + 1u) % 3u][d], got) : 0u;
      }
      if (SCHEME == S_SPARSE && recycle) {
        const uint32_t n_end = batch - count_of(total, KIND);
        if (n_end) {
          g.fbase[sbuf] = atomicAdd(&ctl->free_tail[KIND], n_end);
          atomicAdd(&ctl->ring_tail[(p.it + 1u) % 3u][KIND], n_end);
        }
      }
    }
  }
  word = __shfl_sync(0xFFFFFFFFu, word, 0);
  group_sync(c.group);  // also: all queue entries of the batch have been read

  // position of this thread's outputs among its warp's: survivor; child 0; child 1 (after the warp's
  // children 0 when both go to the same kind)
  const uint32_t r_alive = count_of(word, KIND) + __popc(m_alive & lt_mask);
  const int f0 = k0d ? FD : Q0;             // arrival-word field and destination kind of child 0
  const int d0 = k0d ? int(K_EM) : Q0;
  const uint32_t r_k0 = count_of(word, f0) + __popc((k0d ? m_kd : m_k0) & lt_mask);
  const uint32_t r_k1 = count_of(word, Q1) + ((Q0 == Q1) ? uint32_t(__popc(m_k0)) : 0u) + __popc(m_k1 & lt_mask);
  const int nbuf = int(par ^ 1u);
  constexpr bool kMscVar = (VAR & V_MSC) != 0;
  bool dropped = false;
  c.clk->mark(SEC_ALLOC);
  if (SCHEME == S_DENSE) {
    // A10: whole records into the next arrays
    if (o.alive) {
      const uint32_t dst = g.base[sbuf][KIND] + r_alive;
      if (dst < p.capacity) {
        make_view<L, INSTR>(p, KIND, nbuf, c.cta->probe).store(dst, t);
        if (kMscVar && KIND != K_GAMMA) msc_store(p, KIND, nbuf, dst, t.m0, t.m1, t.m2);
      } else dropped = true;
    }
    if (o.kid[0].kind >= 0) {
      const uint32_t dst = g.base[sbuf][f0] + r_k0;
      if (dst < p.capacity) {
        make_view<L, INSTR>(p, d0, nbuf, c.cta->probe).store(dst, kid_track(t, o.kid[0]));
        if (kMscVar && d0 != K_GAMMA) msc_store(p, d0, nbuf, dst, -1.0f, 0.0f, 0.0f);  // X39: a new track is not initialised
      } else dropped = true;
    }
    if (o.kid[1].kind >= 0) {
      const uint32_t dst = g.base[sbuf][Q1] + r_k1;
      if (dst < p.capacity) {
        make_view<L, INSTR>(p, Q1, nbuf, c.cta->probe).store(dst, kid_track(t, o.kid[1]));
        if (kMscVar && Q1 != K_GAMMA) msc_store(p, Q1, nbuf, dst, -1.0f, 0.0f, 0.0f);
      } else dropped = true;
    }
  } else {
    // A10 sparse: the words the interaction changed, slot pushed onto the next list
    if (o.alive) {
      make_view<L, INSTR>(p, KIND, 0, c.cta->probe).store_changed(slot, t, before_interaction);
      const uint32_t qpos = g.base[sbuf][KIND] + r_alive;
      if (qpos < p.capacity) p.kind[KIND].queue[nbuf][qpos] = slot;
      else dropped = true;
    }
    // slot of the child with rank r among the group's children of field q
    auto child_slot = [&](int q, uint32_t r) -> uint32_t {
      const uint32_t nr = g.rn[sbuf][q];
      if (r < nr) return p.kind[dest_of(q)].free_ring[(g.rbase[sbuf][q] + r) % p.capacity];
      return g.sbase[sbuf][q] + (r - nr);
    };
    if (ends) {
      uint32_t r = uint32_t(__popc(m_end & lt_mask));
      for (int w = 0; w < (gtid >> 5); ++w) r += g.kcnt[sbuf][w];
      p.kind[KIND].free_ring[(g.fbase[sbuf] + r) % p.capacity] = slot;
    }
    if (o.kid[0].kind >= 0) {
      const uint32_t qpos = g.base[sbuf][f0] + r_k0;
      if (r_k0 < g.sgot[sbuf][f0] && qpos < p.capacity) {
        const uint32_t s_new = child_slot(f0, r_k0);
        make_view<L, INSTR>(p, d0, 0, c.cta->probe).store(s_new, kid_track(t, o.kid[0]));
        if (kMscVar && d0 != K_GAMMA) msc_store(p, d0, 0, s_new, -1.0f, 0.0f, 0.0f);
        p.kind[d0].queue[nbuf][qpos] = s_new;
      } else dropped = true;
    }
    if (o.kid[1].kind >= 0) {
      const uint32_t qpos = g.base[sbuf][Q1] + r_k1;
      if (r_k1 < g.sgot[sbuf][Q1] && qpos < p.capacity) {
        const uint32_t s_new = child_slot(Q1, r_k1);
        make_view<L, INSTR>(p, Q1, 0, c.cta->probe).store(s_new, kid_track(t, o.kid[1]));
        if (kMscVar && Q1 != K_GAMMA) msc_store(p, Q1, 0, s_new, -1.0f, 0.0f, 0.0f);
        p.kind[Q1].queue[nbuf][qpos] = s_new;
      } else dropped = true;
    }
  }
  if (dropped) ctl->overflow = 1u;
  c.clk->mark(SEC_STORE);
  return first;
}

// All tiles of one kind that belong to this group, then the left-over parked tracks.
// `first_global_tile` = tiles of the kinds before this one; n_tiles, n_kind are launch-uniform.
template <int L, int SCHEME, bool INSTR, int VAR, int KIND>
__device__ __forceinline__ void run_kind(const Params &p, const Env &env, const GroupRefs &c, uint32_t par,
                                         uint32_t first_global_tile, uint32_t n_tiles, uint32_t n_kind, int &sbuf,
                                         uint32_t &in_phase, uint32_t &tab_phase, int &staged_group) {
  // tiles are dealt round-robin over all groups of the grid, continuing across the kinds
  const uint32_t groups_per_cta = blockDim.x / kGroup;
  const uint32_t n_groups = gridDim.x * groups_per_cta;
  const uint32_t me = blockIdx.x * groups_per_cta + c.group;
  const uint32_t shift = (me + n_groups - first_global_tile % n_groups) % n_groups;
  // a CTA none of whose groups has a tile of this kind skips it altogether -- in particular the
  // CTA-wide staging of the kind's tables (small populations: most CTAs hold one tile of one kind)
  bool cta_has = false;
  for (uint32_t gI = 0; gI < groups_per_cta; ++gI)
    cta_has |= (blockIdx.x * groups_per_cta + gI + n_groups - first_global_tile % n_groups) % n_groups < n_tiles;
  if (!cta_has) return;
  // the group's first tile of this kind is requested before the tables are: the two copies overlap
  // (small populations -- the head and tail of a shower -- are latency-bound, one tile per group)
  if (SCHEME == S_DENSE && shift < n_tiles && c.gtid == 0)  // the staging buffer is free: its last reader passed a barrier
    prefetch_tile<L>(p, KIND, par, shift, n_kind, c.in_buf, &c.g->mbar_in);
  // sparse scheme, direct loads: request the next tile's records into L2 when at least 60 % of the
  // slots handed out so far are live
  bool l2_prefetch = false;
  if (SCHEME == S_SPARSE && !Mapping<L>::kSparseGather) l2_prefetch = 5ull * n_kind >= 3ull * p.ctl->slot_top[KIND];
  if (SCHEME == S_SPARSE && !Mapping<L>::kSparseGather && shift < n_tiles) {  // list entries of the first two tiles
    uint32_t *stash = c.in_buf;
    const uint32_t i0 = shift * kGroup + c.gtid, i1 = i0 + n_groups * kGroup;
    in_phase = 0u;
    if (i0 < n_kind) cp_async_4(static_cast<uint32_t>(__cvta_generic_to_shared(stash + c.gtid)), p.kind[KIND].queue[par] + i0);
    else stash[c.gtid] = kNoSlot;
    if (i1 < n_kind) cp_async_4(static_cast<uint32_t>(__cvta_generic_to_shared(stash + kGroup + c.gtid)), p.kind[KIND].queue[par] + i1);
    else stash[kGroup + c.gtid] = kNoSlot;
    cp_async_commit();
  }
  if (SCHEME == S_SPARSE && Mapping<L>::kSparseGather && shift < n_tiles) {  // each thread: its record of the first tile, its list entry of the second
    const uint32_t i0 = shift * kGroup + c.gtid;
    const uint32_t slot0 = (i0 < n_kind) ? __ldg(&p.kind[KIND].queue[par][i0]) : kNoSlot;
    gather_ahead<L>(p, KIND, par, slot0, i0 + n_groups * kGroup, n_kind, c.in_buf, c.gtid);
  }
  // A3: the cross-section tables of this kind's particle group -> shared memory, one TMA bulk copy
  // (e- and e+ share a group).  CTA-wide: every group is done with the previous tables.
  constexpr int group = (KIND == K_GAMMA) ? 0 : 1;
  if (staged_group != group) {
    __syncthreads();
    // extended physics: the e+ extras (group 2, rule X38) lie behind the e+- group and are staged with it
    const uint32_t stage_bytes = ((VAR & V_PHYS) != 0 && group == 1) ? 2u * p.table_bytes : p.table_bytes;
    if (threadIdx.x == 0) {
      asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
      asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(
                       static_cast<uint32_t>(__cvta_generic_to_shared(&c.cta->mbar))),
                   "r"(stage_bytes)
                   : "memory");
      bulk_g2s(const_cast<float4 *>(env.tab), reinterpret_cast<const unsigned char *>(p.tables) + size_t(group) * p.table_bytes,
               stage_bytes, &c.cta->mbar);
    }
    mbar_wait(&c.cta->mbar, tab_phase);
    tab_phase ^= 1u;
    staged_group = group;
  }
  uint32_t queued = 0u;
  for (uint32_t tile = shift; tile < n_tiles; tile += n_groups) {
    const uint32_t next_tile = (tile + n_groups < n_tiles) ? tile + n_groups : 0xFFFFFFFFu;
    queued = move_tile<L, SCHEME, INSTR, VAR, KIND>(p, env, c, par, tile, next_tile, n_kind, sbuf, in_phase, queued, l2_prefetch);
    sbuf ^= 1;
    if (queued >= uint32_t(kGroup)) {
      queued = interact_batch<L, SCHEME, INSTR, VAR, KIND>(p, env, c, par, queued, sbuf);
      sbuf ^= 1;
    }
  }
  while (queued != 0u) {
    queued = interact_batch<L, SCHEME, INSTR, VAR, KIND>(p, env, c, par, queued, sbuf);
    sbuf ^= 1;
  }
}

// ---------------------------------------------------------------------- the step kernel ------
// Dynamic shared memory: step_smem_bytes() in device_state.cuh.  THREADS = kBlockSmall (4 CTAs/SM)
// or kBlockLarge (one CTA per SM); the code is the same, the number of groups per CTA differs.
#ifndef ADEPT_STEP_MIN_CTAS
#define ADEPT_STEP_MIN_CTAS 4
#endif
template <int L, int SCHEME, bool INSTR, int THREADS, int VAR = 0>
__global__ void __launch_bounds__(THREADS, (THREADS == kBlockSmall) ? ADEPT_STEP_MIN_CTAS : 1) step_kernel(const __grid_constant__ Params p) {
  constexpr int kBlock = THREADS;
  constexpr int kGroupsPerCta = THREADS / kGroup;
  extern __shared__ __align__(128) unsigned char dyn_smem[];
  __shared__ CtaShared sh;
  float4 *s_tab = reinterpret_cast<float4 *>(dyn_smem);
  const int tid = threadIdx.x;
  Ctl *ctl = p.ctl;
  constexpr size_t kInBuf = in_buf_bytes(SCHEME, Mapping<L>::words(kGroup), Mapping<L>::kSparseGather);
  constexpr size_t kPerGroup = kInBuf + queue_bytes(SCHEME, (VAR & V_MSC) != 0);
  GroupRefs c;
  c.cta = &sh;
  c.group = tid / kGroup;
  c.gtid = tid % kGroup;
  c.g = &sh.grp[c.group];
  c.bins.lo = reinterpret_cast<uint32_t *>(dyn_smem + p.table_area);
  c.bins.hi = c.bins.lo + (p.n_slabs + 1u);
  unsigned char *mine = dyn_smem + units_offset(p.table_area, p.n_slabs) + size_t(c.group) * kPerGroup;
  c.in_buf = reinterpret_cast<uint32_t *>(mine);
  c.queue = reinterpret_cast<uint32_t *>(mine + kInBuf);
  SectClock clk;
  c.clk = &clk;

  // Everything that does not depend on the previous launch comes first: with programmatic dependent
  // launch (launch_step) this prologue overlaps the tail of the previous iteration's kernel.
  if (tid == 0) {  // barriers of the asynchronous copies (tables of a particle group, staged tiles)
    mbar_init(&sh.mbar, 1u);
#pragma unroll
    for (int gI = 0; gI < kGroupsPerCta; ++gI) mbar_init(&sh.grp[gI].mbar_in, 1u);
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
  }
  for (uint32_t s = tid; s < 2u * (p.n_slabs + 1u); s += kBlock) c.bins.lo[s] = 0u;  // tally bins, counters
  if (tid < 4) { sh.alive[tid] = 0u; sh.escaped[tid] = 0u; }
  if (tid < kGroupsPerCta) { sh.grp[tid].loaded = 0u; sh.grp[tid].acc[0] = 0u; sh.grp[tid].acc[1] = 0u; }
  if (INSTR) for (int s = tid; s < 3 * kNumFields * 2; s += kBlock) sh.probe[s] = 0u;
  if (tid < kNumSections) sh.sect[tid] = 0u;
  asm volatile("griddepcontrol.wait;" ::: "memory");  // the previous launch has completed and its writes are visible
#ifdef ADEPT_TIMING_SECTIONS
  // launch timeline (timing build): sections[6] += first CTA start -> last CTA end (ns), added when the
  // launch is closed (roll_iterations); sections[kNumSections ..] = scratch {min start, max end} by launch parity
  unsigned long long t_cta_start = 0ull;
  if (tid == 0) {
    asm volatile("mov.u64 %0, %%globaltimer;" : "=l"(t_cta_start));
    atomicMin(&p.sections[kNumSections + 2u * (p.it & 1u)], t_cta_start);
  }
#endif
  // A0: what is alive -- the outputs of the previous launch (complete: it has ended); constant during this launch
  const uint32_t par = p.it & 1u;
  const uint32_t bi = p.it % 3u;
  const uint32_t r0 = ctl->n[bi][0], r1 = ctl->n[bi][1], r2 = ctl->n[bi][2];
  const uint32_t n0 = r0 < p.capacity ? r0 : p.capacity, n1 = r1 < p.capacity ? r1 : p.capacity,
                 n2 = r2 < p.capacity ? r2 : p.capacity;
  // A11 of the previous launch and A0 of this one, off everybody's critical path: first warp of CTA 0
  if (blockIdx.x == 0 && tid < 32) {
#ifdef ADEPT_TIMING_SECTIONS
    roll_iterations<SCHEME == S_SPARSE, (VAR & V_RECYCLE) != 0>(ctl, p.capacity, p.it, true, tid, p.sections);
#else
    roll_iterations<SCHEME == S_SPARSE, (VAR & V_RECYCLE) != 0>(ctl, p.capacity, p.it, true, tid);
#endif
  }
  const uint32_t t0 = (n0 + kGroup - 1) / kGroup, t1 = (n1 + kGroup - 1) / kGroup, t2 = (n2 + kGroup - 1) / kGroup;
  const uint32_t tiles = t0 + t1 + t2;
  __syncthreads();

  if (blockIdx.x * kGroupsPerCta < tiles) {  // CTA-uniform: at least one group of this CTA has a tile
    clk.start(sh.sect, (tid & 31) == 0);

    Env env;
    env.tab = s_tab; env.nodes = p.nodes; env.group_nodes = p.table_bytes / 16u;
    env.ln_e_min = p.ln_e_min; env.inv_dln = p.inv_dln; env.e_cut = p.e_cut;
    env.n_slabs = p.n_slabs; env.abs_mm = p.abs_mm; env.pitch = p.pitch; env.half_xy = p.half_xy;
    env.mat_abs = p.mat_abs; env.mat_gap = p.mat_gap;

    int sbuf = 0;
    uint32_t in_phase = 0u, tab_phase = 0u;
    int staged_group = -1;
    run_kind<L, SCHEME, INSTR, VAR, K_EM>(p, env, c, par, 0u, t0, n0, sbuf, in_phase, tab_phase, staged_group);
    run_kind<L, SCHEME, INSTR, VAR, K_EP>(p, env, c, par, t0, t1, n1, sbuf, in_phase, tab_phase, staged_group);
    run_kind<L, SCHEME, INSTR, VAR, K_GAMMA>(p, env, c, par, t0 + t1, t2, n2, sbuf, in_phase, tab_phase, staged_group);

    // flush the CTA's tallies
    clk.mark(SEC_OTHER);
    __syncthreads();
#ifdef ADEPT_TIMING_SECTIONS
    if (tid < kNumSections && sh.sect[tid]) atomicAdd(&p.sections[tid], static_cast<unsigned long long>(sh.sect[tid]));
#endif
    for (uint32_t s = tid; s <= p.n_slabs; s += kBlock) {
      const unsigned long long v = (static_cast<unsigned long long>(c.bins.hi[s]) << 32) + c.bins.lo[s];
      if (v != 0ull && atomicAdd(&p.tally[s], v) + v < v) ctl->overflow = 1u;  // 2^32 MeV in one bin: reported, not wrapped silently
    }
    if (tid < 3) {
      if (sh.alive[tid]) atomicAdd(&ctl->alive[bi][tid], sh.alive[tid]);
      if (sh.escaped[tid]) atomicAdd(&ctl->esc[bi][tid], sh.escaped[tid]);
    }
    if (INSTR) {
      for (int s = tid; s < 3 * kNumFields * 2; s += kBlock)
        if (sh.probe[s]) atomicAdd(&p.instr_field_rw[s], static_cast<unsigned long long>(sh.probe[s]));
    }
  }

#ifdef ADEPT_TIMING_SECTIONS
  if (tid == 0) {
    unsigned long long t_end;
    asm volatile("mov.u64 %0, %%globaltimer;" : "=l"(t_end));
    atomicMax(&p.sections[kNumSections + 2u * (p.it & 1u) + 1u], t_end);
  }
#endif
}

// ------------------------------------------------------------- host <-> buffer helper kernels --
struct StagedPrimary {  // adept_primary + its global index (rule R4)
  uint32_t kind;
  float pos[3], dir[3], ekin;
  unsigned long long gidx;
};
struct PackedTrack {  // = adept_track, 56 B
  float pos[3], dir[3], ekin, nial[3];
  uint32_t vol, id_lo, id_hi, step;
};

__device__ __forceinline__ Trk unpack(const PackedTrack &a) {
  Trk t;
  t.px = a.pos[0]; t.py = a.pos[1]; t.pz = a.pos[2];
  t.dx = a.dir[0]; t.dy = a.dir[1]; t.dz = a.dir[2];
  t.ekin = a.ekin; t.n0 = a.nial[0]; t.n1 = a.nial[1]; t.n2 = a.nial[2];
  t.vol = a.vol; t.id_lo = a.id_lo; t.id_hi = a.id_hi; t.step = a.step;
  return t;
}
__device__ __forceinline__ PackedTrack pack(const Trk &t) {
  PackedTrack a;
  a.pos[0] = t.px; a.pos[1] = t.py; a.pos[2] = t.pz;
  a.dir[0] = t.dx; a.dir[1] = t.dy; a.dir[2] = t.dz;
  a.ekin = t.ekin; a.nial[0] = t.n0; a.nial[1] = t.n1; a.nial[2] = t.n2;
  a.vol = t.vol; a.id_lo = t.id_lo; a.id_hi = t.id_hi; a.step = t.step;
  return a;
}

template <int L> __device__ __forceinline__ TrackView<L, false> plain_view(const Params &p, int kind, int buf) {
  TrackView<L, false> v;
  v.base = p.kind[kind].rec[buf];
  v.cap = p.capacity;
  v.storage_off = 0; v.buf_index = 0;
  v.kind = kind;
  v.sink.cta_field_rw = nullptr; v.sink.lines = nullptr; v.sink.slots = nullptr;
  return v;
}

// Where entry `i` of the current set of `kind` lives: dense = array index, sparse = slot list.
template <int SCHEME>
__device__ __forceinline__ void place(const Params &p, int kind, uint32_t par, uint32_t entry, uint32_t slot,
                                      int &buf, uint32_t &where) {
  if (SCHEME == S_DENSE) { buf = int(par); where = entry; }
  else { buf = 0; where = slot; p.kind[kind].queue[par][entry] = slot; }
}

// Primaries -> tracks (rule R4 ids, slab located from z; step 0, nial -1).
template <int L, int SCHEME>
__global__ void inject_kernel(const __grid_constant__ Params p, const StagedPrimary *sp, uint32_t n, int kind,
                              uint32_t par, uint32_t entry_base, uint32_t slot_base, unsigned long long seed) {
  const uint32_t i = blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= n) return;
  const StagedPrimary a = sp[i];
  Trk t;
  t.px = a.pos[0]; t.py = a.pos[1]; t.pz = a.pos[2];
  t.dx = a.dir[0]; t.dy = a.dir[1]; t.dz = a.dir[2];
  t.ekin = a.ekin;
  t.n0 = -1.0f; t.n1 = -1.0f; t.n2 = -1.0f;
  int layer = static_cast<int>(a.pos[2] / p.pitch);
  const int last = static_cast<int>(p.n_slabs / 2u) - 1;
  if (layer > last) layer = last;
  const float rel = a.pos[2] - static_cast<float>(layer) * p.pitch;
  t.vol = 2u * static_cast<uint32_t>(layer) + ((rel >= p.abs_mm) ? 1u : 0u);
  const uint2 id = primary_id(a.gidx, seed);
  t.id_lo = id.x; t.id_hi = id.y;
  t.step = 0u;
  int buf; uint32_t where;
  place<SCHEME>(p, kind, par, entry_base + i, slot_base + i, buf, where);
  plain_view<L>(p, kind, buf).store(where, t);
  if (p.physics == 2u && kind != K_GAMMA) msc_store(p, kind, buf, where, -1.0f, 0.0f, 0.0f);  // X39: not initialised
}

template <int L, int SCHEME>
__global__ void load_kernel(const __grid_constant__ Params p, const PackedTrack *src, const uint32_t *slots,
                            uint32_t n, int kind, uint32_t par, uint32_t entry_base, uint32_t slot_base) {
  const uint32_t i = blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= n) return;
  const PackedTrack a = src[i];
  // preconditions of adept_load_tracks (include/adept.h): the step kernel indexes the slab geometry and
  // the tally bins by `vol`, packs the pending interaction into the top bits of `step`, and divides by
  // the direction cosines
  const bool finite = isfinite(a.pos[0]) && isfinite(a.pos[1]) && isfinite(a.pos[2]) && isfinite(a.dir[0]) &&
                      isfinite(a.dir[1]) && isfinite(a.dir[2]) && !isnan(a.nial[0]) && !isnan(a.nial[1]) &&
                      !isnan(a.nial[2]);
  const bool moving = a.dir[0] != 0.0f || a.dir[1] != 0.0f || a.dir[2] != 0.0f;
  const bool energy = (a.ekin >= p.e_cut && a.ekin <= p.e_max) || (kind == K_EP && a.ekin >= 0.0f && a.ekin < p.e_cut);
  if (!(finite && moving && energy && a.vol < p.n_slabs && a.step < (1u << 20))) {
    p.ctl->bad_input = 1u;
    return;
  }
  int buf; uint32_t where;
  place<SCHEME>(p, kind, par, entry_base + i, slots ? slots[i] : slot_base + i, buf, where);
  plain_view<L>(p, kind, buf).store(where, unpack(a));
  if (p.physics == 2u && kind != K_GAMMA) msc_store(p, kind, buf, where, -1.0f, 0.0f, 0.0f);  // X39: not initialised
}

template <int L, int SCHEME>
__global__ void read_kernel(const __grid_constant__ Params p, PackedTrack *dst, uint32_t first, uint32_t n,
                            int kind, uint32_t par) {
  const uint32_t i = blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= n) return;
  const uint32_t entry = first + i;
  if (SCHEME == S_DENSE) dst[i] = pack(plain_view<L>(p, kind, int(par)).load(entry));
  else dst[i] = pack(plain_view<L>(p, kind, 0).load(p.kind[kind].queue[par][entry]));
}

// ----------------------------------------------------------------- per-layout entry points ----
// One table of launchers per layout; adept_api.cu picks the table once at adept_create.  (Layout,
// scheme and instrumentation are compile-time parameters of every kernel.)
struct LayoutOps {
  size_t (*record_words)(size_t capacity);
  bool sparse_gather;  // Mapping<L>::kSparseGather
  int (*step_ctas_per_sm)(int scheme, int instr, int variant, int threads, size_t dyn_smem);
  cudaError_t (*launch_step)(int scheme, int instr, const Params &, int threads, unsigned grid, size_t dyn_smem,
                             cudaStream_t);  // Params::recycle / physics pick the kernel variant
  cudaError_t (*launch_inject)(int scheme, const Params &, const void *staged, uint32_t n, int kind, uint32_t par,
                               uint32_t entry_base, uint32_t slot_base, unsigned long long seed, cudaStream_t);
  cudaError_t (*launch_load)(int scheme, const Params &, const void *staged, const uint32_t *slots, uint32_t n,
                             int kind, uint32_t par, uint32_t entry_base, uint32_t slot_base, cudaStream_t);
  cudaError_t (*launch_read)(int scheme, const Params &, void *staged, uint32_t first, uint32_t n, int kind,
                             uint32_t par, cudaStream_t);
};

// cudaFuncAttributeMaxDynamicSharedMemorySize is a property of (device, kernel instantiation), shared
// by every context of the process: keep a running maximum and never lower it, so that a later context
// with smaller tables cannot break the launches of an earlier, larger one.
inline cudaError_t ensure_dynamic_smem(const void *kernel, size_t bytes) {
  static std::mutex mu;
  static std::map<std::pair<int, const void *>, size_t> granted;
  int dev = 0;
  cudaError_t e = cudaGetDevice(&dev);
  if (e != cudaSuccess) return e;
  std::lock_guard<std::mutex> lock(mu);
  size_t &have = granted[std::make_pair(dev, kernel)];
  if (bytes <= have) return cudaSuccess;
  e = cudaFuncSetAttribute(kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, int(bytes));
  if (e == cudaSuccess) have = bytes;
  return e;
}

template <int L> struct OpsImpl {
  // The extended physics is instantiated for the plain (non-counting) kernels without slot recycling.
  template <int T, typename F> static auto pick_t(int scheme, int instr, int var, F f) {
    if (var & V_MSC)
      return scheme == S_DENSE ? f(step_kernel<L, S_DENSE, false, T, V_PHYS | V_MSC>) : f(step_kernel<L, S_SPARSE, false, T, V_PHYS | V_MSC>);
    if (var & V_PHYS)
      return scheme == S_DENSE ? f(step_kernel<L, S_DENSE, false, T, V_PHYS>) : f(step_kernel<L, S_SPARSE, false, T, V_PHYS>);
    if (scheme == S_DENSE) return instr ? f(step_kernel<L, S_DENSE, true, T>) : f(step_kernel<L, S_DENSE, false, T>);
    if (var & V_RECYCLE) return instr ? f(step_kernel<L, S_SPARSE, true, T, V_RECYCLE>) : f(step_kernel<L, S_SPARSE, false, T, V_RECYCLE>);
    return instr ? f(step_kernel<L, S_SPARSE, true, T>) : f(step_kernel<L, S_SPARSE, false, T>);
  }
  template <typename F> static auto pick(int scheme, int instr, int var, int threads, F f) {
    return threads == kBlockLarge ? pick_t<kBlockLarge>(scheme, instr, var, f) : pick_t<kBlockSmall>(scheme, instr, var, f);
  }
  static size_t record_words(size_t cap) { return Mapping<L>::words(cap); }
  static int step_ctas_per_sm(int scheme, int instr, int var, int threads, size_t dyn) {
    return pick(scheme, instr, var, threads, [&](auto *k) {
      int n = 0;
      if (ensure_dynamic_smem(reinterpret_cast<const void *>(k), dyn) != cudaSuccess) return -1;
      if (cudaOccupancyMaxActiveBlocksPerMultiprocessor(&n, k, threads, dyn) != cudaSuccess) return -1;
      return n;
    });
  }
  static cudaError_t launch_step(int scheme, int instr, const Params &p, int threads, unsigned grid, size_t dyn,
                                 cudaStream_t s) {
    return pick(scheme, instr, (p.recycle ? V_RECYCLE : 0) | (p.physics ? V_PHYS : 0) | (p.physics == 2u ? V_MSC : 0), threads, [&](auto *k) {
      const cudaError_t e = ensure_dynamic_smem(reinterpret_cast<const void *>(k), dyn);
      if (e != cudaSuccess) return e;
      // Programmatic dependent launch: the CTAs of this launch may become resident, and run their
      // prologue up to griddepcontrol.wait, while the previous kernel of the stream is still finishing
      // (its slowest CTA alone) -- iterations of small populations are a chain of
      // latencies, and this takes the launch latency out of it.
      cudaLaunchConfig_t cfg = {};
      cfg.gridDim = dim3(grid);
      cfg.blockDim = dim3(unsigned(threads));
      cfg.dynamicSmemBytes = dyn;
      cfg.stream = s;
      cudaLaunchAttribute attr[1];
      attr[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
      attr[0].val.programmaticStreamSerializationAllowed = 1;
      cfg.attrs = attr;
#ifdef ADEPT_NO_PDL   // experiment builds only (build.py extra_flags): plain stream-ordered launches
      cfg.numAttrs = 0u;
#else
      cfg.numAttrs = 1u;
#endif
      return cudaLaunchKernelEx(&cfg, k, p);
    });
  }
  static cudaError_t launch_inject(int scheme, const Params &p, const void *staged, uint32_t n, int kind,
                                   uint32_t par, uint32_t eb, uint32_t sb, unsigned long long seed, cudaStream_t s) {
    const unsigned g = (n + 255) / 256;
    const StagedPrimary *sp = static_cast<const StagedPrimary *>(staged);
    if (scheme == S_DENSE) inject_kernel<L, S_DENSE><<<g, 256, 0, s>>>(p, sp, n, kind, par, eb, sb, seed);
    else inject_kernel<L, S_SPARSE><<<g, 256, 0, s>>>(p, sp, n, kind, par, eb, sb, seed);
    return cudaGetLastError();
  }
  static cudaError_t launch_load(int scheme, const Params &p, const void *staged, const uint32_t *slots, uint32_t n,
                                 int kind, uint32_t par, uint32_t eb, uint32_t sb, cudaStream_t s) {
    const unsigned g = (n + 255) / 256;
    const PackedTrack *src = static_cast<const PackedTrack *>(staged);
    if (scheme == S_DENSE) load_kernel<L, S_DENSE><<<g, 256, 0, s>>>(p, src, slots, n, kind, par, eb, sb);
    else load_kernel<L, S_SPARSE><<<g, 256, 0, s>>>(p, src, slots, n, kind, par, eb, sb);
    return cudaGetLastError();
  }
  static cudaError_t launch_read(int scheme, const Params &p, void *staged, uint32_t first, uint32_t n, int kind,
                                 uint32_t par, cudaStream_t s) {
    const unsigned g = (n + 255) / 256;
    PackedTrack *dst = static_cast<PackedTrack *>(staged);
    if (scheme == S_DENSE) read_kernel<L, S_DENSE><<<g, 256, 0, s>>>(p, dst, first, n, kind, par);
    else read_kernel<L, S_SPARSE><<<g, 256, 0, s>>>(p, dst, first, n, kind, par);
    return cudaGetLastError();
  }
  static LayoutOps make() {
    return LayoutOps{record_words, Mapping<L>::kSparseGather, step_ctas_per_sm, launch_step, launch_inject, launch_load, launch_read};
  }
};

extern const LayoutOps kOpsAoS, kOpsSoA, kOpsAoSoA32, kOpsAoSoA64, kOpsSoA16, kOpsAoSoA16, kOpsAoSoA128, kOpsHC16, kOpsAoSoA8;

}  // namespace adept
