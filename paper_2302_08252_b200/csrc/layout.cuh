// Track record and its compile-time switchable memory layout.
//
// The paper separates "the algorithmic view of data from its mapping to device memory" (LLAMA,
// PAPER.md:25, 35): kernels address a field of a track, a mapping chosen at compile time turns
// (slot, field) into an address — AoS, SoA or AoSoA-n ("AABBCCAABBCC" for n = 2) —
// and instrumented mappings count accesses per field (Trace/FieldAccessCount)
// and per byte/row (Heatmap).  This header is that idea reduced to what the
// step needs: `Mapping<L>` is pure index arithmetic with no run-time state, `TrackView<L, INSTR>`
// moves whole records or single words between registers and memory, and `Probe` is the counting
// hook compiled in only for the instrumented build.
//
// Record = 14 four-byte words, word order = adept_track (include/adept.h).
#pragma once
#include <cstdint>
#include <cuda_runtime.h>

namespace adept {

enum Field : int {
  F_PX = 0, F_PY, F_PZ, F_DX, F_DY, F_DZ, F_EKIN, F_N0, F_N1, F_N2, F_VOL, F_IDLO, F_IDHI, F_STEP,
  kNumFields = 14
};
enum LayoutId : int { L_AOS = 0, L_SOA = 1, L_AOSOA32 = 2, L_AOSOA64 = 3, L_SOA16 = 4, L_AOSOA16 = 5, L_AOSOA128 = 6,
                      L_HC16 = 7, L_AOSOA8 = 8 };

// A track in registers.
struct Trk {
  float px, py, pz, dx, dy, dz, ekin, n0, n1, n2;
  uint32_t vol, id_lo, id_hi, step;
  // rule X39 (physics 2, e+- only): InitialRange (< 0 = not initialised), DynamicRangeFactor, TlimitMin.
  // Not part of the 14-word record: they live in the kind's side array (KindStorage::msc).
  float m0, m1, m2;
};

__device__ __forceinline__ uint32_t trk_word(const Trk &t, int f) {
  switch (f) {
    case F_PX: return __float_as_uint(t.px);
    case F_PY: return __float_as_uint(t.py);
    case F_PZ: return __float_as_uint(t.pz);
    case F_DX: return __float_as_uint(t.dx);
    case F_DY: return __float_as_uint(t.dy);
    case F_DZ: return __float_as_uint(t.dz);
    case F_EKIN: return __float_as_uint(t.ekin);
    case F_N0: return __float_as_uint(t.n0);
    case F_N1: return __float_as_uint(t.n1);
    case F_N2: return __float_as_uint(t.n2);
    case F_VOL: return t.vol;
    case F_IDLO: return t.id_lo;
    case F_IDHI: return t.id_hi;
    default: return t.step;
  }
}

__device__ __forceinline__ void trk_set_word(Trk &t, int f, uint32_t w) {
  switch (f) {
    case F_PX: t.px = __uint_as_float(w); break;
    case F_PY: t.py = __uint_as_float(w); break;
    case F_PZ: t.pz = __uint_as_float(w); break;
    case F_DX: t.dx = __uint_as_float(w); break;
    case F_DY: t.dy = __uint_as_float(w); break;
    case F_DZ: t.dz = __uint_as_float(w); break;
    case F_EKIN: t.ekin = __uint_as_float(w); break;
    case F_N0: t.n0 = __uint_as_float(w); break;
    case F_N1: t.n1 = __uint_as_float(w); break;
    case F_N2: t.n2 = __uint_as_float(w); break;
    case F_VOL: t.vol = w; break;
    case F_IDLO: t.id_lo = w; break;
    case F_IDHI: t.id_hi = w; break;
    default: t.step = w; break;
  }
}

// ---- mappings: (capacity, slot, field) -> word index inside one record buffer ---------------
// Capacities are multiples of 128 slots (one tile), so every SoA field array and every AoSoA block
// starts on a 128-byte line.
template <int L> struct Mapping;
// Mapping<L>::kSparseGather: the sparse scheme fetches this layout's records one tile ahead by
// asynchronous 16-byte copies (step_impl.cuh gather_record); false = direct loads.

template <> struct Mapping<L_AOS> {  // 14 words padded to 16: one record = 64 B = 2 sectors = 4 x 16 B
  static constexpr int kStride = 16;
  static constexpr bool kSparseGather = true;
  __host__ __device__ static constexpr size_t words(size_t cap) { return cap * kStride; }
  __host__ __device__ static constexpr size_t index(size_t, size_t slot, int f, int = 0) { return slot * kStride + f; }
};
template <> struct Mapping<L_SOA> {  // 14 arrays of `cap` words
  static constexpr bool kSparseGather = false;
  __host__ __device__ static constexpr size_t words(size_t cap) { return cap * kNumFields; }
  __host__ __device__ static constexpr size_t index(size_t cap, size_t slot, int f, int = 0) { return f * cap + slot; }
};
template <int N> struct AoSoAMapping {  // blocks of N tracks, field-major inside a block (N * 56 B)
  static constexpr int kLanes = N;
  static constexpr bool kSparseGather = false;
  __host__ __device__ static constexpr size_t words(size_t cap) { return cap * kNumFields; }
  __host__ __device__ static constexpr size_t index(size_t, size_t slot, int f, int = 0) {
    return (slot / kLanes) * (kLanes * kNumFields) + f * kLanes + (slot % kLanes);
  }
};
template <> struct Mapping<L_AOSOA32> : AoSoAMapping<32> {};  // "AoSoA-n"
template <> struct Mapping<L_AOSOA64> : AoSoAMapping<64> {};  // the paper's fastest
template <> struct Mapping<L_AOSOA16> : AoSoAMapping<16> {};  // "several lane counts"
template <> struct Mapping<L_AOSOA128> : AoSoAMapping<128> {};  // one block per tile
template <> struct Mapping<L_AOSOA8> : AoSoAMapping<8> {};  // the shortest lane count of SURVEY.md §8(f) item 2: a block is 448 B, a field run one sector
// SoA of 16-byte field groups (SURVEY.md §8(f) item 1 "grouped-SoA of 16-byte vectors"; BASELINE.json
// north_star "coalesced, vectorised 16-byte loads of SoA fields"): four arrays of `cap` vectors --
// {pos.xyz, dir.x}, {dir.y, dir.z, ekin, nial.0}, {nial.1, nial.2, vol, id_lo} (16 B each) and
// {id_hi, step} (8 B) -- so that a record moves with four vector instructions instead of fourteen and
// consecutive slots are consecutive vectors.
template <> struct Mapping<L_SOA16> {
  static constexpr bool kSparseGather = false;  // measured: faster only above ~80 % occupancy
  __host__ __device__ static constexpr size_t words(size_t cap) { return cap * kNumFields; }
  __host__ __device__ static constexpr size_t index(size_t cap, size_t slot, int f, int = 0) {
    return (f < 12) ? size_t(f / 4) * 4 * cap + slot * 4 + (f % 4) : 12 * cap + slot * 2 + (f - 12);
  }
};
// Hot/cold split with per-kind grouping ("Individualizing,
// splitting and regrouping ... A separation of hot and cold data would be a first step ... different
// layouts per particle type"): the SoA16 geometry -- three arrays of 16-byte vectors and one of
// 8-byte vectors -- with the record's words regrouped by how the step of each particle kind uses them:
//   vector A (hot, rewritten every step)   {pos.x, pos.y, pos.z, step}                 all kinds
//   vector B (hot, rewritten every step)   gamma: {nial.0, nial.1, nial.2, vol}   e+-: {ekin, nial.0, nial.1, vol}
//   vector C (read; written by an interaction only)  gamma: {dir.x, dir.y, dir.z, ekin}   e+-: {dir.x, dir.y, dir.z, nial.2}
//   vector D (cold: read only when a draw is made)   {id_lo, id_hi}
// In the sparse single buffer the move half of a step then rewrites 32 bytes of a record (A and B)
// instead of 56-64.  `kind` = 2 (gamma) selects the first grouping.
template <> struct Mapping<L_HC16> {
  static constexpr bool kSparseGather = false;
  __host__ __device__ static constexpr size_t words(size_t cap) { return cap * kNumFields; }
  __host__ __device__ static constexpr int position(int f, int kind) {
    constexpr int kGamma[kNumFields] = {0, 1, 2, 8, 9, 10, 11, 4, 5, 6, 7, 12, 13, 3};
    constexpr int kElec[kNumFields] = {0, 1, 2, 8, 9, 10, 4, 5, 6, 11, 7, 12, 13, 3};
    return kind == 2 ? kGamma[f] : kElec[f];
  }
  __host__ __device__ static constexpr size_t index(size_t cap, size_t slot, int f, int kind = 2) {
    return Mapping<L_SOA16>::index(cap, slot, position(f, kind));
  }
};

// ---- L_HC16: a record <-> its four vectors, by particle kind ----------------------------------
__device__ __forceinline__ void hc16_pack(bool gamma, const Trk &t, uint4 &a, uint4 &b, uint4 &c, uint2 &d) {
  a = make_uint4(__float_as_uint(t.px), __float_as_uint(t.py), __float_as_uint(t.pz), t.step);
  if (gamma) {
    b = make_uint4(__float_as_uint(t.n0), __float_as_uint(t.n1), __float_as_uint(t.n2), t.vol);
    c = make_uint4(__float_as_uint(t.dx), __float_as_uint(t.dy), __float_as_uint(t.dz), __float_as_uint(t.ekin));
  } else {
    b = make_uint4(__float_as_uint(t.ekin), __float_as_uint(t.n0), __float_as_uint(t.n1), t.vol);
    c = make_uint4(__float_as_uint(t.dx), __float_as_uint(t.dy), __float_as_uint(t.dz), __float_as_uint(t.n2));
  }
  d = make_uint2(t.id_lo, t.id_hi);
}
__device__ __forceinline__ Trk hc16_unpack(bool gamma, const uint4 &a, const uint4 &b, const uint4 &c, const uint2 &d) {
  Trk t;
  t.px = __uint_as_float(a.x); t.py = __uint_as_float(a.y); t.pz = __uint_as_float(a.z); t.step = a.w;
  t.dx = __uint_as_float(c.x); t.dy = __uint_as_float(c.y); t.dz = __uint_as_float(c.z);
  if (gamma) {
    t.n0 = __uint_as_float(b.x); t.n1 = __uint_as_float(b.y); t.n2 = __uint_as_float(b.z);
    t.ekin = __uint_as_float(c.w);
  } else {
    t.ekin = __uint_as_float(b.x); t.n0 = __uint_as_float(b.y); t.n1 = __uint_as_float(b.z);
    t.n2 = __uint_as_float(c.w);
  }
  t.vol = b.w;
  t.id_lo = d.x; t.id_hi = d.y;
  return t;
}

// ---- access counting (instrumented build only) -----------------------------------------------
// field_rw: shared-memory counters [14][2] of the CTA (flushed once per kernel);
// lines / slots: global counters of the kind's record storage (line = 128 B, "row").
struct ProbeSink {
  uint32_t *cta_field_rw;  // shared
  uint32_t *lines;         // global, indexed by (byte offset in the kind's record storage) / 128
  uint32_t *slots;         // global, indexed by buffer_index * capacity + slot
};

template <bool INSTR> struct Probe {
  __device__ __forceinline__ void touch(const ProbeSink &, int, int, size_t, size_t) const {}
};
template <> struct Probe<true> {
  __device__ __forceinline__ void touch(const ProbeSink &s, int field, int is_write, size_t byte_off,
                                        size_t slot_index) const {
    atomicAdd(&s.cta_field_rw[field * 2 + is_write], 1u);
    atomicAdd(&s.lines[byte_off >> 7], 1u);
    atomicAdd(&s.slots[slot_index], 1u);
  }
};

// ---- view of one record buffer ----------------------------------------------------------------
template <int L, bool INSTR> struct TrackView {
  uint32_t *base;      // first word of this buffer
  uint32_t cap;        // slots
  size_t storage_off;  // byte offset of this buffer inside the kind's record storage (probe only)
  uint32_t buf_index;  // 0/1 (probe only)
  int kind;            // particle kind of the buffer (per-kind layouts)
  ProbeSink sink;

  using Map = Mapping<L>;

  __device__ __forceinline__ void probe(int f, int w, size_t slot) const {
    Probe<INSTR>().touch(sink, f, w, storage_off + Map::index(cap, slot, f, kind) * 4, size_t(buf_index) * cap + slot);
  }

  __device__ __forceinline__ uint32_t load_word(uint32_t slot, int f) const {
    probe(f, 0, slot);
    return base[Map::index(cap, slot, f, kind)];
  }
  __device__ __forceinline__ void store_word(uint32_t slot, int f, uint32_t w) const {
    probe(f, 1, slot);
    base[Map::index(cap, slot, f, kind)] = w;
  }

  // whole record -> registers
  __device__ __forceinline__ Trk load(uint32_t slot) const {
    Trk t;
    if constexpr (L == L_HC16) {
      using V = Mapping<L_SOA16>;
      const uint4 a = *reinterpret_cast<const uint4 *>(base + V::index(cap, slot, 0));
      const uint4 b = *reinterpret_cast<const uint4 *>(base + V::index(cap, slot, 4));
      const uint4 c = *reinterpret_cast<const uint4 *>(base + V::index(cap, slot, 8));
      const uint2 d = *reinterpret_cast<const uint2 *>(base + V::index(cap, slot, 12));
      t = hc16_unpack(kind == 2, a, b, c, d);
      if constexpr (INSTR) {
#pragma unroll
        for (int f = 0; f < kNumFields; ++f) probe(f, 0, slot);
      }
    } else if constexpr (L == L_AOS || L == L_SOA16) {
      uint4 a, b, c;
      uint2 d;
      if constexpr (L == L_AOS) {
        const uint4 *r = reinterpret_cast<const uint4 *>(base + size_t(slot) * Map::kStride);
        a = r[0]; b = r[1]; c = r[2];
        d = *reinterpret_cast<const uint2 *>(r + 3);
      } else {
        a = *reinterpret_cast<const uint4 *>(base + Map::index(cap, slot, 0));
        b = *reinterpret_cast<const uint4 *>(base + Map::index(cap, slot, 4));
        c = *reinterpret_cast<const uint4 *>(base + Map::index(cap, slot, 8));
        d = *reinterpret_cast<const uint2 *>(base + Map::index(cap, slot, 12));
      }
      t.px = __uint_as_float(a.x); t.py = __uint_as_float(a.y); t.pz = __uint_as_float(a.z);
      t.dx = __uint_as_float(a.w); t.dy = __uint_as_float(b.x); t.dz = __uint_as_float(b.y);
      t.ekin = __uint_as_float(b.z); t.n0 = __uint_as_float(b.w);
      t.n1 = __uint_as_float(c.x); t.n2 = __uint_as_float(c.y);
      t.vol = c.z; t.id_lo = c.w; t.id_hi = d.x; t.step = d.y;
      if constexpr (INSTR) {
#pragma unroll
        for (int f = 0; f < kNumFields; ++f) probe(f, 0, slot);
      }
    } else {
#pragma unroll
      for (int f = 0; f < kNumFields; ++f) trk_set_word(t, f, load_word(slot, f));
    }
    return t;
  }

  // registers -> whole record
  __device__ __forceinline__ void store(uint32_t slot, const Trk &t) const {
    if constexpr (L == L_HC16) {
      using V = Mapping<L_SOA16>;
      uint4 a, b, c;
      uint2 d;
      hc16_pack(kind == 2, t, a, b, c, d);
      *reinterpret_cast<uint4 *>(base + V::index(cap, slot, 0)) = a;
      *reinterpret_cast<uint4 *>(base + V::index(cap, slot, 4)) = b;
      *reinterpret_cast<uint4 *>(base + V::index(cap, slot, 8)) = c;
      *reinterpret_cast<uint2 *>(base + V::index(cap, slot, 12)) = d;
      if constexpr (INSTR) {
#pragma unroll
        for (int f = 0; f < kNumFields; ++f) probe(f, 1, slot);
      }
    } else if constexpr (L == L_AOS || L == L_SOA16) {
      const uint4 a = make_uint4(__float_as_uint(t.px), __float_as_uint(t.py), __float_as_uint(t.pz), __float_as_uint(t.dx));
      const uint4 b = make_uint4(__float_as_uint(t.dy), __float_as_uint(t.dz), __float_as_uint(t.ekin), __float_as_uint(t.n0));
      const uint4 c = make_uint4(__float_as_uint(t.n1), __float_as_uint(t.n2), t.vol, t.id_lo);
      if constexpr (L == L_AOS) {
        uint4 *r = reinterpret_cast<uint4 *>(base + size_t(slot) * Map::kStride);
        r[0] = a; r[1] = b; r[2] = c;
        r[3] = make_uint4(t.id_hi, t.step, 0u, 0u);  // tail padding written so that sectors are whole
      } else {
        *reinterpret_cast<uint4 *>(base + Map::index(cap, slot, 0)) = a;
        *reinterpret_cast<uint4 *>(base + Map::index(cap, slot, 4)) = b;
        *reinterpret_cast<uint4 *>(base + Map::index(cap, slot, 8)) = c;
        *reinterpret_cast<uint2 *>(base + Map::index(cap, slot, 12)) = make_uint2(t.id_hi, t.step);
      }
      if constexpr (INSTR) {
#pragma unroll
        for (int f = 0; f < kNumFields; ++f) probe(f, 1, slot);
      }
    } else {
#pragma unroll
      for (int f = 0; f < kNumFields; ++f) store_word(slot, f, trk_word(t, f));
    }
  }

  // registers -> the words the move half of a step assigns (sparse single buffer: in-place update,
  // PAPER.md:115 "writes concentrated on ..."): pos, nial of the kind's processes, step -- and ekin
  // for e+-, vol when the step crossed into another slab.  dir never changes in the move half, ids
  // never.  A word assigned the value it already had (a zero-length step) is written again; the
  // counting build uses store_changed below instead and counts only real changes.
  // N1: e+- also assign nial[1] (extended physics, rule X36); N2: e+ also nial[2] (rule X38); DIR: e+-
  // also the direction (multiple scattering, rule X39).
  template <bool GAMMA, bool N1 = false, bool N2 = false, bool DIR = false> __device__ __forceinline__ void store_moved(uint32_t slot, const Trk &t, bool vol_changed) const {
    if constexpr (L == L_HC16) {
      // the two hot vectors; e+ under the extended physics also assigns nial[2], which lives in vector C
      using V = Mapping<L_SOA16>;
      uint4 a, b, c;
      uint2 d;
      hc16_pack(GAMMA, t, a, b, c, d);
      *reinterpret_cast<uint4 *>(base + V::index(cap, slot, 0)) = a;
      *reinterpret_cast<uint4 *>(base + V::index(cap, slot, 4)) = b;
      if constexpr (N2 || DIR) *reinterpret_cast<uint4 *>(base + V::index(cap, slot, 8)) = c;
      (void)vol_changed; (void)d;
    } else if constexpr (L == L_AOS || L == L_SOA16) {
      // 16-byte pieces {pos, dir.x} {dir.yz, ekin, nial0} {nial12, vol, id_lo} {id_hi, step}: a photon
      // rewrites all four, e+- three and the third only with vol
      uint4 *q0, *q1, *q2;
      uint2 *q3;
      if constexpr (L == L_AOS) {
        uint4 *r = reinterpret_cast<uint4 *>(base + size_t(slot) * Map::kStride);
        q0 = r; q1 = r + 1; q2 = r + 2; q3 = reinterpret_cast<uint2 *>(r + 3);
      } else {
        q0 = reinterpret_cast<uint4 *>(base + Map::index(cap, slot, 0));
        q1 = reinterpret_cast<uint4 *>(base + Map::index(cap, slot, 4));
        q2 = reinterpret_cast<uint4 *>(base + Map::index(cap, slot, 8));
        q3 = reinterpret_cast<uint2 *>(base + Map::index(cap, slot, 12));
      }
      *q0 = make_uint4(__float_as_uint(t.px), __float_as_uint(t.py), __float_as_uint(t.pz), __float_as_uint(t.dx));
      *q1 = make_uint4(__float_as_uint(t.dy), __float_as_uint(t.dz), __float_as_uint(t.ekin), __float_as_uint(t.n0));
      if (GAMMA || N1 || vol_changed) *q2 = make_uint4(__float_as_uint(t.n1), __float_as_uint(t.n2), t.vol, t.id_lo);
      *q3 = make_uint2(t.id_hi, t.step);
    } else {
      base[Map::index(cap, slot, F_PX)] = __float_as_uint(t.px);
      base[Map::index(cap, slot, F_PY)] = __float_as_uint(t.py);
      base[Map::index(cap, slot, F_PZ)] = __float_as_uint(t.pz);
      base[Map::index(cap, slot, F_N0)] = __float_as_uint(t.n0);
      if constexpr (GAMMA) {
        base[Map::index(cap, slot, F_N1)] = __float_as_uint(t.n1);
        base[Map::index(cap, slot, F_N2)] = __float_as_uint(t.n2);
      } else {
        base[Map::index(cap, slot, F_EKIN)] = __float_as_uint(t.ekin);
        if constexpr (N1) base[Map::index(cap, slot, F_N1)] = __float_as_uint(t.n1);
        if constexpr (N2) base[Map::index(cap, slot, F_N2)] = __float_as_uint(t.n2);
        if constexpr (DIR) {
          base[Map::index(cap, slot, F_DX)] = __float_as_uint(t.dx);
          base[Map::index(cap, slot, F_DY)] = __float_as_uint(t.dy);
          base[Map::index(cap, slot, F_DZ)] = __float_as_uint(t.dz);
        }
      }
      if (vol_changed) base[Map::index(cap, slot, F_VOL)] = t.vol;
      base[Map::index(cap, slot, F_STEP)] = t.step;
    }
  }

  // registers -> only the words that differ from `old` (sparse single buffer: in-place update)
  __device__ __forceinline__ void store_changed(uint32_t slot, const Trk &t, const Trk &old) const {
    if constexpr (L == L_HC16 && !INSTR) {
      using V = Mapping<L_SOA16>;
      uint4 a, b, c, oa, ob, oc;
      uint2 d, od;
      hc16_pack(kind == 2, t, a, b, c, d);
      hc16_pack(kind == 2, old, oa, ob, oc, od);
      auto ne = [](const uint4 &x, const uint4 &y) { return x.x != y.x || x.y != y.y || x.z != y.z || x.w != y.w; };
      if (ne(a, oa)) *reinterpret_cast<uint4 *>(base + V::index(cap, slot, 0)) = a;
      if (ne(b, ob)) *reinterpret_cast<uint4 *>(base + V::index(cap, slot, 4)) = b;
      if (ne(c, oc)) *reinterpret_cast<uint4 *>(base + V::index(cap, slot, 8)) = c;
      if (d.x != od.x || d.y != od.y) *reinterpret_cast<uint2 *>(base + V::index(cap, slot, 12)) = d;
      return;
    }
    if constexpr ((L == L_AOS || L == L_SOA16) && !INSTR) {
      // layouts that keep a record's words in 16-byte pieces: a piece with a changed word is rewritten
      // whole (the thread owns the record; the unchanged words of the piece are written back as they
      // are), so an update costs two to four vector stores instead of seven to fourteen scalar ones.
      // The counting build below keeps the word-by-word form: it counts the words the step changes.
      auto differ = [&](int f) { return trk_word(t, f) != trk_word(old, f); };  // bit patterns, as below
      const bool c0 = differ(F_PX) || differ(F_PY) || differ(F_PZ) || differ(F_DX);
      const bool c1 = differ(F_DY) || differ(F_DZ) || differ(F_EKIN) || differ(F_N0);
      const bool c2 = differ(F_N1) || differ(F_N2) || differ(F_VOL) || differ(F_IDLO);
      const bool c3 = differ(F_IDHI) || differ(F_STEP);
      uint4 *q0, *q1, *q2;
      uint2 *q3;
      if constexpr (L == L_AOS) {
        uint4 *r = reinterpret_cast<uint4 *>(base + size_t(slot) * Map::kStride);
        q0 = r; q1 = r + 1; q2 = r + 2; q3 = reinterpret_cast<uint2 *>(r + 3);
      } else {
        q0 = reinterpret_cast<uint4 *>(base + Map::index(cap, slot, 0));
        q1 = reinterpret_cast<uint4 *>(base + Map::index(cap, slot, 4));
        q2 = reinterpret_cast<uint4 *>(base + Map::index(cap, slot, 8));
        q3 = reinterpret_cast<uint2 *>(base + Map::index(cap, slot, 12));
      }
      if (c0) *q0 = make_uint4(__float_as_uint(t.px), __float_as_uint(t.py), __float_as_uint(t.pz), __float_as_uint(t.dx));
      if (c1) *q1 = make_uint4(__float_as_uint(t.dy), __float_as_uint(t.dz), __float_as_uint(t.ekin), __float_as_uint(t.n0));
      if (c2) *q2 = make_uint4(__float_as_uint(t.n1), __float_as_uint(t.n2), t.vol, t.id_lo);
      if (c3) *q3 = make_uint2(t.id_hi, t.step);
      return;
    }
#pragma unroll
    for (int f = 0; f < kNumFields; ++f) {
      const uint32_t w = trk_word(t, f);
      if (w != trk_word(old, f)) store_word(slot, f, w);
    }
  }
};

}  // namespace adept
