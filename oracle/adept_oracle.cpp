// ============================================================================
// ORACLE — TEST INFRASTRUCTURE, NOT THE PRODUCT.
//
// A plain, slow, single-threaded CPU transport of the simplified AdePT
// electromagnetic step (e-, e+, gamma) that the CUDA library in
// paper_2302_08252_b200/ must reproduce.  Only tests/, __graft_entry__.smoke()
// and bench.py's cpu_baseline / --impl reference legs may build, load or call
// it.  It shares no source, header, table or constant generator with the CUDA
// path and neither includes the other.
//
// What it follows.  The paper (arXiv 2302.08252, /root/reference/PAPER.md)
// fixes only the *structure* of the hot path:
//   * per-particle-type lists of active tracks, one transport pass per
//     iteration, survivors and secondaries handed to the next iteration
//     (§2; Fig. 1);
//   * the track record's fields: RNG state, energy, three "number of
//     interaction lengths left", position, direction, navigation state
//     (Fig. 3);
//   * secondaries initialised from the parent's position and navigation state
//     (Fig. 2);
//   * 50 alternating absorber/gap box layers and the energy deposit per layer
//     as the result (§4); batches of primaries.
// The physics content is BASELINE.json's north_star/configs ("samples the
// physics step from log-grid cross-section tables, takes the geometry step to
// the next slab boundary, applies continuous energy loss and discrete
// interactions, emits secondaries"; Philox-4x32 keyed by (track id, step, draw
// index)).  Every point on which those two sources are silent is a numbered
// reading in DESIGN.md §3 (rules R1-R6, M7-M11, T12-T14, S16-S31, X35-X39); the code
// below follows those rules one by one, in their order and notation, with no
// blocking, fusion or reordering.
//
// Pins (tests/test_oracle_*.py, all `-m "not gpu"`): Philox known-answer
// vectors; exhaustive u01 grid; lg/ex/sincos2pi against libm in double; table
// lookup on ln-linear tables; narrow-beam attenuation exp(-mu x) (exact count
// by stream enumeration, brute-force probability over the whole u grid,
// statistical); 1-track/1-slab brute force over the u grid; geometry walks;
// per-event energy conservation; <T(x)> = T0 exp(-x/X0) for brems; Compton
// energy-momentum conservation and Compton edge; CSDA range; pair/photo
// branch energies; lockstep == depth-first order independence.
// Extended physics (tables.physics = 1; DESIGN.md rules X35-X39, SURVEY.md
// §8(f) item 3): delta-ray production on nial[1] of e+- (X36), the Compton
// energy fraction from the full Klein-Nishina distribution by composition and
// rejection (X37), annihilation in flight on nial[2] of e+ (X38), multiple
// scattering with three more words per e+- track (X39, tables.physics = 2).
// Pins (tests/test_oracle_extended.py): the eps distribution against quadrature of the textbook Klein-Nishina density (KS distance, mean);
// the delta-ray energy against the closed-form 1/T^2 CDF; exact two-body
// energy-momentum closure; S_restricted + int T dSigma_delta = S; per-event
// energy conservation; lockstep == depth-first; X38: two-photon energy and
// momentum closure, uniform k1, Heitler's limits; X39: the closed-form step
// limit on constant tables, exponential 1 - cos(theta), re-initialisation at a face.
// Parity unpinned (no external closed form exists): the full-shower
// longitudinal profile — only sanity checks (P-table).
//
// Arithmetic contract (M7): every track quantity is IEEE-754 binary32,
// round-to-nearest-even, no contraction except where fmaf() is written;
// compile with -O2 -ffp-contract=off and without -ffast-math.  Tallies are
// fp64 sums of fp32 terms.
// ============================================================================
#include <cmath>
#include <cstdint>
#include <cstring>
#include <array>
#include <limits>
#include <unordered_map>
#include <vector>

namespace {

// ------------------------------------------------------------------ types --
struct Track {            // 14 four-byte words, 56 B
  float pos[3];
  float dir[3];
  float ekin;
  float nial[3];          // "NumIALeft.0-2"
  uint32_t vol;           // navigation state = slab index
  uint32_t id_lo, id_hi;  // counter-RNG key
  uint32_t step;          // counter-RNG counter
};
static_assert(sizeof(Track) == 56, "track record is 56 bytes");

struct Primary { uint32_t kind; float pos[3], dir[3], ekin; };
static_assert(sizeof(Primary) == 32, "primary record is 32 bytes");

struct Geometry {
  uint32_t n_layers;
  float abs_mm, gap_mm, half_xy_mm;
  uint32_t mat_abs, mat_gap;
};

struct TablesIn {          // as passed over the C interface
  uint32_t n_bins, n_materials;
  float e_min, e_max, ln_e_min, inv_dln, e_cut;
  const float *data;       // [mat][group][qty][n_bins+1]
  uint32_t physics;        // rule X35: 0 = rules S16-S32, 1 = with the extended rules X36-X38, 2 = also X39
  const float *data_x;     // physics >= 1: [mat][3][n_bins+1]: Sigma_delta of e+- (X36), Sigma_annihilation of e+ (X38),
                           // transport cross-section Sigma_tr of e+- (X39) [1/mm]
};

struct Result {
  uint64_t live[3], steps[3], secondaries[3], killed[3], escaped_n[3];
  uint64_t slots_used[3];
  uint64_t iterations;
  double e_injected, e_escaped;
  double e_escaped_kind[3];   // diagnostic split of e_escaped (sums to it)
};

struct TraceRec {          // one per processed track when tracing is on
  uint32_t id_lo, id_hi, step, kind;
  int32_t winner;          // -2 annihilation at rest, -1 GEOM, 3 ELOSS, 0..2 process
  float margin;            // smallest relative gap of any threshold decision taken
};

enum { KIND_EM = 0, KIND_EP = 1, KIND_GAMMA = 2 };
enum { GROUP_GAMMA = 0, GROUP_ELEC = 1 };
enum { W_ANNIH = -2, W_GEOM = -1, W_ELOSS = 3, W_MSC = 5 };
enum { FACE_ZP = 0, FACE_ZM = 1, FACE_XY = 2 };

const float INF = std::numeric_limits<float>::infinity();

// -------------------------------------------------- R1: Philox-4x32-10 -----
// Salmon, Moraes, Dror, Shaw, "Parallel random numbers: as easy as 1, 2, 3",
// SC'11.  BASELINE.json: "draws the same Philox-4x32 random streams keyed by
// (track id, step, draw index)".
void philox4x32_10(const uint32_t ctr[4], const uint32_t key[2], uint32_t out[4]) {
  uint32_t c0 = ctr[0], c1 = ctr[1], c2 = ctr[2], c3 = ctr[3];
  uint32_t k0 = key[0], k1 = key[1];
  for (int round = 0; round < 10; ++round) {
    const uint64_t p0 = (uint64_t)0xD2511F53u * (uint64_t)c0;
    const uint64_t p1 = (uint64_t)0xCD9E8D57u * (uint64_t)c2;
    const uint32_t n0 = (uint32_t)(p1 >> 32) ^ c1 ^ k0;
    const uint32_t n1 = (uint32_t)p1;
    const uint32_t n2 = (uint32_t)(p0 >> 32) ^ c3 ^ k1;
    const uint32_t n3 = (uint32_t)p0;
    c0 = n0; c1 = n1; c2 = n2; c3 = n3;
    k0 += 0x9E3779B9u;
    k1 += 0xBB67AE85u;
  }
  out[0] = c0; out[1] = c1; out[2] = c2; out[3] = c3;
}

// R3: u32 -> uniform on the odd 24-bit grid, never 0 or 1, exact.
float u01(uint32_t x) {
  return (float)(2u * (x >> 9) + 1u) * 5.9604644775390625e-08f;   // 2^-24
}

// ------------------------------------------------------ M8-M10: maths ------
uint32_t f2u(float f) { uint32_t u; std::memcpy(&u, &f, 4); return u; }
float u2f(uint32_t u) { float f; std::memcpy(&f, &u, 4); return f; }

const float LN2_HI = 0.693145751953125f;        // 0x3F317200
const float LN2_LO = 1.428606765330187e-06f;    // fl32(ln 2 - LN2_HI) = 0x35BFBE8E

// M8: ln m = 2 atanh((m-1)/(m+1)), m in (1/sqrt2, sqrt2]
float lg(float x) {
  const uint32_t b = f2u(x);
  int e = (int)((b >> 23) & 0xFFu) - 127;
  const uint32_t mb = b & 0x7FFFFFu;
  float m = u2f(mb | 0x3F800000u);
  if (mb > 0x3504F3u) { m = m * 0.5f; e += 1; }
  const float s = (m - 1.0f) / (m + 1.0f);
  const float s2 = s * s;
  float p = 1.0f / 11.0f;
  p = fmaf(p, s2, 1.0f / 9.0f);
  p = fmaf(p, s2, 1.0f / 7.0f);
  p = fmaf(p, s2, 1.0f / 5.0f);
  p = fmaf(p, s2, 1.0f / 3.0f);
  p = p * s2;
  const float r = fmaf(p, s, s);
  const float r2 = r + r;
  const float ef = (float)e;
  return fmaf(ef, LN2_HI, fmaf(ef, LN2_LO, r2));
}

// M9: exp by range reduction to |r| <= ln2/2 and a degree-7 Taylor polynomial
float ex(float x) {
  const float k = rintf(x * 1.4426950408889634f);
  float r = fmaf(-k, LN2_HI, x);
  r = fmaf(-k, LN2_LO, r);
  float p = 1.0f / 5040.0f;
  p = fmaf(p, r, 1.0f / 720.0f);
  p = fmaf(p, r, 1.0f / 120.0f);
  p = fmaf(p, r, 1.0f / 24.0f);
  p = fmaf(p, r, 1.0f / 6.0f);
  p = fmaf(p, r, 0.5f);
  p = fmaf(p, r, 1.0f);
  p = fmaf(p, r, 1.0f);
  const int ki = (int)k;
  return u2f(f2u(p) + ((uint32_t)ki << 23));      // p * 2^k through the exponent bits
}

// M10: (sin, cos)(2 pi u), u in (0, 1)
void sincos2pi(float u, float *sn, float *cs) {
  const float q = rintf(4.0f * u);
  const float t = fmaf(-0.25f, q, u);             // exact
  const float a = t * 6.283185307179586f;
  const float a2 = a * a;
  float p = -1.0f / 39916800.0f;
  p = fmaf(p, a2, 1.0f / 362880.0f);
  p = fmaf(p, a2, -1.0f / 5040.0f);
  p = fmaf(p, a2, 1.0f / 120.0f);
  p = fmaf(p, a2, -1.0f / 6.0f);
  const float s = fmaf(p * a2, a, a);
  float c = -1.0f / 3628800.0f;
  c = fmaf(c, a2, 1.0f / 40320.0f);
  c = fmaf(c, a2, -1.0f / 720.0f);
  c = fmaf(c, a2, 1.0f / 24.0f);
  c = fmaf(c, a2, -0.5f);
  c = fmaf(c, a2, 1.0f);
  switch (((int)q) & 3) {
    case 0: *sn = s;  *cs = c;  break;
    case 1: *sn = c;  *cs = -s; break;
    case 2: *sn = -s; *cs = -c; break;
    default: *sn = -c; *cs = s; break;
  }
}

// --------------------------------------------------------- T13: lookup -----
struct Tables {
  uint32_t n_bins = 0, n_materials = 0;
  float e_min = 0, e_max = 0, ln_e_min = 0, inv_dln = 0, e_cut = 0;
  std::vector<float> data;
  uint32_t physics = 0;       // X35
  std::vector<float> data_x;  // X36: Sigma_delta per material
  const float *q(uint32_t mat, int group, int qty) const {
    return data.data() + ((size_t)(mat * 2 + group) * 3 + qty) * (n_bins + 1);
  }
  const float *qx(uint32_t mat, int which) const { return data_x.data() + ((size_t)mat * 3 + which) * (n_bins + 1); }
};

struct Bin { int j; float f; };

Bin locate_bin(const Tables &t, float lnE) {
  const float x = (lnE - t.ln_e_min) * t.inv_dln;
  int j = (int)x;
  if (j < 0) j = 0;
  if (j > (int)t.n_bins - 1) j = (int)t.n_bins - 1;
  Bin b;
  b.j = j;
  b.f = x - (float)j;
  return b;
}

float interp(const float *T, Bin b) {
  return fmaf(b.f, T[b.j + 1] - T[b.j], T[b.j]);
}

// ------------------------------------------------------ S27: rotation ------
void rotate(const float d[3], float st, float ct, float sphi, float cphi, float out[3]) {
  const float q2 = fmaf(-d[2], d[2], 1.0f);
  float o0, o1, o2;
  if (q2 > 1e-10f) {
    const float sp = sqrtf(q2);
    const float ux = ((d[0] * d[2]) * cphi - d[1] * sphi) / sp;
    const float uy = ((d[1] * d[2]) * cphi + d[0] * sphi) / sp;
    const float uz = -(sp * cphi);
    o0 = fmaf(st, ux, ct * d[0]);
    o1 = fmaf(st, uy, ct * d[1]);
    o2 = fmaf(st, uz, ct * d[2]);
  } else {
    o0 = st * cphi;
    o1 = st * sphi;
    o2 = (d[2] < 0.0f) ? -ct : ct;
  }
  const float nn = sqrtf(fmaf(o0, o0, fmaf(o1, o1, o2 * o2)));
  out[0] = o0 / nn;
  out[1] = o1 / nn;
  out[2] = o2 / nn;
}

// ----------------------------------------------------------- the oracle ----
struct Oracle {
  Geometry geo{};
  Tables tab;
  uint64_t seed = 0;
  float pitch = 0, mc2 = 0.51099895f, two_mc2 = 0;
  std::vector<Track> cur[3], nxt[3];
  std::vector<double> edep;       // per slab, 2*n_layers
  Result res{};
  uint64_t next_primary = 0;
  bool tracing = false;
  std::vector<TraceRec> trace;
  std::vector<Primary> pending;
  // X39: the three multiple-scattering words of an e+- track (the paper's InitialRange,
  // DynamicRangeFactor, TlimitMin), by track id; a track without an entry has
  // InitialRange = -1 (not initialised).  They are not part of the 14-word record.
  std::unordered_map<uint64_t, std::array<float, 3>> msc;

  float zlo(uint32_t i) const {   // S21 / DESIGN §4 geometry
    return fmaf((float)(i >> 1), pitch, (i & 1u) ? geo.abs_mm : 0.0f);
  }
};

struct Rng {                       // R2: lazy, fixed-purpose draws (calls 3..18: the tries of rule X37)
  uint32_t key[2];
  uint32_t step;
  bool have[19] = {};
  uint32_t blk[19][4];
  uint32_t word(int call, int w) {
    if (!have[call]) {
      const uint32_t ctr[4] = {step, (uint32_t)call, 0u, 0u};
      philox4x32_10(ctr, key, blk[call]);
      have[call] = true;
    }
    return blk[call][w];
  }
  float u(int call, int w) { return u01(word(call, w)); }
};

struct Child { int kind; Track t; };

inline void note_margin(float &margin, float a, float b) {
  // relative gap between two compared quantities (for the decision-margin report)
  const float den = fmaxf(fmaxf(fabsf(a), fabsf(b)), 1e-30f);
  if (std::isfinite(a) && std::isfinite(b)) {
    const float g = fabsf(a - b) / den;
    if (g < margin) margin = g;
  }
}

// S28/R5/R6: a secondary starts at the parent's position and slab
// (PAPER.md:47-60 InitAsSecondary(parentPos, parentNavState)), step 0, nial -1,
// id = words (2*ordinal, 2*ordinal+1) of call 2 of the parent's stream.
Track make_child(const Track &parent, Rng &rng, int ordinal, const float dir[3], float ekin) {
  Track c;
  for (int i = 0; i < 3; ++i) { c.pos[i] = parent.pos[i]; c.dir[i] = dir[i]; c.nial[i] = -1.0f; }
  c.ekin = ekin;
  c.vol = parent.vol;
  c.id_lo = rng.word(2, 2 * ordinal);
  c.id_hi = rng.word(2, 2 * ordinal + 1);
  c.step = 0;
  return c;
}

// One call = one track, one iteration (rules S16-S27, S31).  Returns true if
// the track survives into the next iteration.  `t` is updated in place.
bool step_track(Oracle &o, int kind, Track &t, Child children[2], int &n_children) {
  const Tables &tab = o.tab;
  const float e_cut = tab.e_cut;
  n_children = 0;
  Rng rng;
  rng.key[0] = t.id_lo; rng.key[1] = t.id_hi; rng.step = t.step;
  o.res.steps[kind] += 1;
  float margin = INF;
  int winner_out = W_GEOM;
  auto finish = [&](bool alive) {
    if (o.tracing) o.trace.push_back(TraceRec{t.id_lo, t.id_hi, rng.step, (uint32_t)kind, winner_out, margin});
    for (int i = 0; i < n_children; ++i) o.res.secondaries[children[i].kind] += 1;
    if (!alive) o.res.killed[kind] += 1;
    return alive;
  };
  auto deposit = [&](uint32_t slab, float e) { o.edep[slab] += (double)e; };

  // S17: positron below the cut annihilates at rest, first.
  if (kind == KIND_EP) note_margin(margin, t.ekin, e_cut);
  if (kind == KIND_EP && t.ekin < e_cut) {
    winner_out = W_ANNIH;
    deposit(t.vol, t.ekin);
    const float ct = 1.0f - 2.0f * rng.u(1, 2);
    const float st = sqrtf(fmaf(-ct, ct, 1.0f));
    float sphi, cphi;
    sincos2pi(rng.u(1, 3), &sphi, &cphi);
    const float d0[3] = {st * cphi, st * sphi, ct};
    const float d1[3] = {-d0[0], -d0[1], -d0[2]};
    children[0].kind = KIND_GAMMA; children[0].t = make_child(t, rng, 0, d0, o.mc2);
    children[1].kind = KIND_GAMMA; children[1].t = make_child(t, rng, 1, d1, o.mc2);
    n_children = 2;
    return finish(false);
  }

  const bool extended = tab.physics >= 1u;                       // X35
  const bool with_msc = tab.physics == 2u && kind != KIND_GAMMA;  // X39
  const uint64_t track_key = ((uint64_t)t.id_hi << 32) | t.id_lo;
  float m[3] = {-1.0f, 0.0f, 0.0f};
  if (with_msc) {
    auto it = o.msc.find(track_key);
    if (it != o.msc.end()) { m[0] = it->second[0]; m[1] = it->second[1]; m[2] = it->second[2]; o.msc.erase(it); }
  }
  auto keep_msc = [&]() { if (with_msc) o.msc[track_key] = {m[0], m[1], m[2]}; };
  // X36: e+- process 1 = delta-ray production; X38: e+ process 2 = annihilation in flight
  const int NP = (kind == KIND_GAMMA) ? 3 : (extended ? (kind == KIND_EP ? 3 : 2) : 1);
  const int group = (kind == KIND_GAMMA) ? GROUP_GAMMA : GROUP_ELEC;

  // S18: re-sample spent interaction lengths.
  for (int j = 0; j < NP; ++j)
    if (t.nial[j] <= 0.0f) t.nial[j] = -lg(rng.u(0, j));

  // S19: cross sections at the pre-step energy and material.
  const uint32_t vol0 = t.vol;
  const uint32_t mat = (vol0 & 1u) ? o.geo.mat_gap : o.geo.mat_abs;
  const float E0 = t.ekin;
  const Bin bin = locate_bin(tab, lg(E0));
  float sig[3] = {0.0f, 0.0f, 0.0f};
  float sj[3] = {INF, INF, INF};
  for (int j = 0; j < NP; ++j) {
    sig[j] = (kind != KIND_GAMMA && j >= 1) ? interp(tab.qx(mat, j - 1), bin)   // X36: Sigma_delta, X38: Sigma_annihilation
                                            : interp(tab.q(mat, group, j), bin);
    sj[j] = (sig[j] > 0.0f) ? t.nial[j] / sig[j] : INF;
  }

  // S20: continuous-loss step limit (e+- only).
  float R = 0.0f, S0 = 0.0f, s_e = INF;
  if (kind != KIND_GAMMA) {
    S0 = interp(tab.q(mat, GROUP_ELEC, 1), bin);
    R = interp(tab.q(mat, GROUP_ELEC, 2), bin);
    const float r_min = 0.1f, f_r = 0.2f;
    if (R <= r_min) {
      s_e = R;
    } else {
      const float fr = f_r * R;
      s_e = (fr > r_min) ? fr : r_min;
    }
  }

  // S21: distance to the slab faces and to the transverse box.
  const float z_lo = o.zlo(vol0), z_hi = o.zlo(vol0 + 1u);
  // X39a, X39b: multiple-scattering step limit max(DynamicRangeFactor * InitialRange, TlimitMin),
  // (re-)initialised at the start of a track and after every slab crossing
  float sig_tr = 0.0f, s_m = INF;
  if (with_msc) {
    sig_tr = interp(tab.qx(mat, 2), bin);
    if (sig_tr > 0.0f) {
      if (m[0] < 0.0f) {
        float safety = fminf(t.pos[2] - z_lo, z_hi - t.pos[2]);
        if (!(safety > 0.0f)) safety = 0.0f;
        m[0] = R;
        m[1] = fmaxf(0.04f, (0.6f * safety) / R);
        m[2] = fmaxf(1e-3f, 0.01f / sig_tr);
      }
      s_m = fmaxf(m[1] * m[0], m[2]);
    }
  }
  const float H = o.geo.half_xy_mm;
  const float dx = t.dir[0], dy = t.dir[1], dz = t.dir[2];
  const float s_z = (dz > 0.0f) ? (z_hi - t.pos[2]) / dz : (dz < 0.0f) ? (z_lo - t.pos[2]) / dz : INF;
  const float s_x = (dx > 0.0f) ? (H - t.pos[0]) / dx : (dx < 0.0f) ? (-H - t.pos[0]) / dx : INF;
  const float s_y = (dy > 0.0f) ? (H - t.pos[1]) / dy : (dy < 0.0f) ? (-H - t.pos[1]) / dy : INF;
  float s_g = s_z;
  int face = (dz > 0.0f) ? FACE_ZP : FACE_ZM;
  note_margin(margin, s_x, s_g);
  if (s_x < s_g) { s_g = s_x; face = FACE_XY; }
  note_margin(margin, s_y, s_g);
  if (s_y < s_g) { s_g = s_y; face = FACE_XY; }
  if (!(s_g > 0.0f)) s_g = 0.0f;

  // S22: winner, strict '<' so ties go to the earlier candidate.
  float s = s_g;
  int w = W_GEOM;
  if (kind != KIND_GAMMA) {
    note_margin(margin, s_e, s);
    if (s_e < s) { s = s_e; w = W_ELOSS; }
    if (with_msc) {
      note_margin(margin, s_m, s);
      if (s_m < s) { s = s_m; w = W_MSC; }
    }
  }
  for (int j = 0; j < NP; ++j) {
    note_margin(margin, sj[j], s);
    if (sj[j] < s) { s = sj[j]; w = j; }
  }
  winner_out = w;

  // S23: move.
  for (int c = 0; c < 3; ++c) t.pos[c] = fmaf(s, t.dir[c], t.pos[c]);
  for (int j = 0; j < NP; ++j) t.nial[j] = fmaf(-s, sig[j], t.nial[j]);
  t.step = rng.step + 1u;

  // S24: continuous loss and scoring (e+- only).
  if (kind != KIND_GAMMA) {
    float E_post;
    if (w == W_ELOSS) note_margin(margin, s, R);
    if (w == W_ELOSS && s >= R) {
      E_post = 0.0f;
    } else {
      float E_mid = fmaf(-0.5f * s, S0, E0);
      if (!(E_mid > e_cut)) E_mid = e_cut;
      const float S_mid = interp(tab.q(mat, GROUP_ELEC, 1), locate_bin(tab, lg(E_mid)));
      float dE = s * S_mid;
      if (!(dE < E0)) dE = E0;
      E_post = E0 - dE;
    }
    deposit(vol0, E0 - E_post);
    note_margin(margin, E_post, e_cut);
    if (E_post < e_cut) {
      if (kind == KIND_EM) { deposit(vol0, E_post); return finish(false); }
      t.ekin = E_post;                // e+: kept alive for S17 at its next step
      keep_msc();
      return finish(true);
    }
    t.ekin = E_post;
    // X39c: deflection by multiple scattering along the step, 1 - cos(theta) exponential with mean s Sigma_tr
    if (with_msc && sig_tr > 0.0f && s > 0.0f) {
      const float tau = s * sig_tr;
      float c = fmaf(tau, lg(rng.u(3, 0)), 1.0f);
      if (c < -1.0f) c = -1.0f;
      const float sn = sqrtf(fmaf(-c, c, 1.0f));
      float sphi, cphi;
      sincos2pi(rng.u(3, 1), &sphi, &cphi);
      float d1[3];
      rotate(t.dir, sn, c, sphi, cphi, d1);
      for (int i = 0; i < 3; ++i) t.dir[i] = d1[i];
    }
  }

  // S25: boundary crossing / escape.
  if (w == W_GEOM) {
    bool escape = false;
    if (face == FACE_ZP) {
      t.pos[2] = z_hi;
      if (vol0 + 1u >= 2u * o.geo.n_layers) escape = true; else { t.vol = vol0 + 1u; m[0] = -1.0f; }  // X39d
    } else if (face == FACE_ZM) {
      t.pos[2] = z_lo;
      if (vol0 == 0u) escape = true; else { t.vol = vol0 - 1u; m[0] = -1.0f; }  // X39d
    } else {
      escape = true;
    }
    if (escape) {
      const double e_out = (double)t.ekin + ((kind == KIND_EP) ? (double)o.two_mc2 : 0.0);
      o.res.e_escaped += e_out;
      o.res.e_escaped_kind[kind] += e_out;
      o.res.escaped_n[kind] += 1;
      return finish(false);
    }
  } else if (w != W_ELOSS && w != W_MSC) {
    // S26: discrete interaction of process w.
    t.nial[w] = -1.0f;
    if (kind == KIND_EP && w == 2) {
      // X38: annihilation in flight on an electron at rest: two photons, isotropic in the centre-of-
      // momentum frame, boosted to the laboratory; the positron dies
      const float E = t.ekin;
      const float e_tot = E + o.two_mc2;
      const float pp = sqrtf(E * e_tot);                   // positron momentum, p^2 = E (E + 2 mc^2)
      const float beta = pp / e_tot;                       // velocity of the centre of momentum
      const float cs = 1.0f - 2.0f * rng.u(1, 2);
      const float k1 = (0.5f * e_tot) * fmaf(beta, cs, 1.0f);
      const float k2 = e_tot - k1;
      float c1 = (cs + beta) / fmaf(beta, cs, 1.0f);
      if (c1 > 1.0f) c1 = 1.0f;
      if (c1 < -1.0f) c1 = -1.0f;
      const float s1 = sqrtf(fmaf(-c1, c1, 1.0f));
      float sphi, cphi;
      sincos2pi(rng.u(1, 3), &sphi, &cphi);
      float d1[3];
      rotate(t.dir, s1, c1, sphi, cphi, d1);
      float q[3];
      for (int c = 0; c < 3; ++c) q[c] = fmaf(pp, t.dir[c], -(k1 * d1[c]));
      const float qn = sqrtf(fmaf(q[0], q[0], fmaf(q[1], q[1], q[2] * q[2])));
      note_margin(margin, k1, e_cut);
      if (k1 >= e_cut) {
        children[n_children].kind = KIND_GAMMA; children[n_children].t = make_child(t, rng, 0, d1, k1);
        ++n_children;
      } else {
        deposit(vol0, k1);
      }
      note_margin(margin, k2, e_cut);
      if (k2 >= e_cut && qn > 0.0f) {
        const float d2[3] = {q[0] / qn, q[1] / qn, q[2] / qn};
        children[n_children].kind = KIND_GAMMA; children[n_children].t = make_child(t, rng, 1, d2, k2);
        ++n_children;
      } else {
        deposit(vol0, k2);
      }
      return finish(false);
    } else if (kind != KIND_GAMMA && w == 1) {
      // X36: delta-ray production (the 1/T^2 term common to Moller and Bhabha scattering) on
      // [e_cut, E/2], two-body kinematics on a free electron at rest
      // X36 guard: the interaction happens at the POST-step energy, which continuous loss may have taken
      // to or below 2 e_cut although Sigma_delta (looked up at the pre-step energy, and interpolated across
      // the bin that holds 2 e_cut) was positive.  The spectrum's interval [e_cut, E/2] is then empty: no
      // delta ray is made and the track goes on unchanged (nial[1] is spent and re-sampled at its next step).
      const float E = t.ekin;
      const float a = e_cut, b = 0.5f * E;
      note_margin(margin, b, a);
      if (b > a) {
        float T = (a * b) / (b - rng.u(1, 0) * (b - a));
        if (!(T > a)) T = a;
        if (!(T < b)) T = b;
        const float E1 = E - T;
        const float tau = E + o.two_mc2;
        float cd = sqrtf((T * tau) / (E * (T + o.two_mc2)));
        float cp = sqrtf((E1 * tau) / (E * (E1 + o.two_mc2)));
        if (cd > 1.0f) cd = 1.0f;
        if (cp > 1.0f) cp = 1.0f;
        const float sd = sqrtf(fmaf(-cd, cd, 1.0f));
        const float sp = sqrtf(fmaf(-cp, cp, 1.0f));
        float sphi, cphi;
        sincos2pi(rng.u(1, 1), &sphi, &cphi);
        float dd[3], dp[3];
        rotate(t.dir, sd, cd, sphi, cphi, dd);
        rotate(t.dir, sp, cp, -sphi, -cphi, dp);
        children[0].kind = KIND_EM; children[0].t = make_child(t, rng, 0, dd, T);
        n_children = 1;
        t.ekin = E1;
        for (int c = 0; c < 3; ++c) t.dir[c] = dp[c];
      }
    } else if (kind != KIND_GAMMA) {
      // bremsstrahlung, 1/k spectrum on [e_cut, E]
      const float E = t.ekin;
      float k = e_cut * ex(rng.u(1, 0) * lg(E / e_cut));
      if (!(k < E)) k = E;
      children[0].kind = KIND_GAMMA; children[0].t = make_child(t, rng, 0, t.dir, k);
      n_children = 1;
      const float E_new = E - k;
      note_margin(margin, E_new, e_cut);
      if (E_new < e_cut) {
        if (kind == KIND_EM) { deposit(vol0, E_new); return finish(false); }
      }
      t.ekin = E_new;
    } else if (w == 0) {
      // pair production, uniform split of E - 2 mc^2
      const float E_av = t.ekin - o.two_mc2;
      const float T_minus = rng.u(1, 0) * E_av;
      const float T_plus = E_av - T_minus;
      note_margin(margin, T_minus, e_cut);
      if (T_minus >= e_cut) {
        children[n_children].kind = KIND_EM; children[n_children].t = make_child(t, rng, 0, t.dir, T_minus);
        ++n_children;
      } else {
        deposit(vol0, T_minus);
      }
      children[n_children].kind = KIND_EP; children[n_children].t = make_child(t, rng, 1, t.dir, T_plus);
      ++n_children;
      return finish(false);
    } else if (w == 1) {
      // Compton, 1/eps spectrum on [1/(1+2k), 1] with exact kinematics
      const float E = t.ekin;
      const float kappa = E / o.mc2;
      const float L = lg(fmaf(2.0f, kappa, 1.0f));
      float eps;
      if (!extended) {
        eps = ex(-(rng.u(1, 0) * L));
      } else {
        // X37: eps from the Klein-Nishina distribution f(eps) ~ (1/eps + eps)(1 - eps sin^2/(1 + eps^2))
        // by composition and rejection (try k draws call 3 + k, words 0..2; at most 16 tries)
        const float eps0 = 1.0f / fmaf(2.0f, kappa, 1.0f);
        const float eps0sq = eps0 * eps0;
        const float a1 = L;                              // ln(1/eps0)
        const float a2 = 0.5f * (1.0f - eps0sq);
        const float thr = a1 / (a1 + a2);
        eps = 1.0f;
        for (int k = 0; k < 16; ++k) {
          const float u1 = rng.u(3 + k, 0), u2 = rng.u(3 + k, 1), u3 = rng.u(3 + k, 2);
          if (thr > u1) eps = ex(-(a1 * u2));
          else eps = sqrtf(fmaf(1.0f - eps0sq, u2, eps0sq));
          if (eps < eps0) eps = eps0;
          if (eps > 1.0f) eps = 1.0f;
          const float tt = (1.0f - eps) / (kappa * eps);
          const float sin2 = tt * (2.0f - tt);
          const float g = 1.0f - (eps * sin2) / fmaf(eps, eps, 1.0f);
          if (g >= u3) break;
        }
      }
      const float E1 = eps * E;
      const float T = E - E1;
      float ct = 1.0f - (((1.0f / eps) - 1.0f) / kappa);
      if (ct > 1.0f) ct = 1.0f;
      if (ct < -1.0f) ct = -1.0f;
      const float st = sqrtf(fmaf(-ct, ct, 1.0f));
      float sphi, cphi;
      sincos2pi(rng.u(1, 1), &sphi, &cphi);
      float d1[3];
      rotate(t.dir, st, ct, sphi, cphi, d1);
      float p[3];
      for (int c = 0; c < 3; ++c) p[c] = fmaf(E, t.dir[c], -(E1 * d1[c]));
      const float pn = sqrtf(fmaf(p[0], p[0], fmaf(p[1], p[1], p[2] * p[2])));
      note_margin(margin, T, e_cut);
      if (T >= e_cut && pn > 0.0f) {
        const float de[3] = {p[0] / pn, p[1] / pn, p[2] / pn};
        children[0].kind = KIND_EM; children[0].t = make_child(t, rng, 0, de, T);
        n_children = 1;
      } else {
        deposit(vol0, T);
      }
      note_margin(margin, E1, e_cut);
      if (E1 < e_cut) {
        deposit(vol0, E1);
        return finish(false);
      }
      t.ekin = E1;
      for (int c = 0; c < 3; ++c) t.dir[c] = d1[c];
    } else {
      // photoelectric absorption: e- with T = E along dir
      children[0].kind = KIND_EM; children[0].t = make_child(t, rng, 0, t.dir, t.ekin);
      n_children = 1;
      return finish(false);
    }
  }
  // S31: runaway guard (never expected).
  if (t.step >= (1u << 20)) {
    deposit(t.vol, t.ekin);
    if (kind == KIND_EP) deposit(t.vol, o.two_mc2);
    return finish(false);
  }
  keep_msc();
  return finish(true);
}

// S28: lockstep — iteration n steps every track alive at its start exactly once.
void iterate(Oracle &o) {
  Child ch[2];
  for (int kind = 0; kind < 3; ++kind) {
    for (Track &t : o.cur[kind]) {
      int nc = 0;
      if (step_track(o, kind, t, ch, nc)) o.nxt[kind].push_back(t);
      for (int i = 0; i < nc; ++i) o.nxt[ch[i].kind].push_back(ch[i].t);
    }
  }
  for (int kind = 0; kind < 3; ++kind) {
    o.cur[kind].swap(o.nxt[kind]);
    o.nxt[kind].clear();
    o.res.live[kind] = o.cur[kind].size();
    if (o.cur[kind].size() > o.res.slots_used[kind]) o.res.slots_used[kind] = o.cur[kind].size();
  }
  o.res.iterations += 1;
}

// Order-independence check: follow each track (and then its children) to the
// end before touching the next one.  Must give the same integers and tallies.
void run_depth_first(Oracle &o) {
  std::vector<Child> stack;
  for (int kind = 2; kind >= 0; --kind) {
    for (size_t i = o.cur[kind].size(); i-- > 0;) stack.push_back(Child{kind, o.cur[kind][i]});
    o.cur[kind].clear();
  }
  Child ch[2];
  while (!stack.empty()) {
    Child c = stack.back();
    stack.pop_back();
    for (;;) {
      int nc = 0;
      const bool alive = step_track(o, c.kind, c.t, ch, nc);
      for (int i = 0; i < nc; ++i) stack.push_back(ch[i]);
      if (!alive) break;
    }
  }
  for (int kind = 0; kind < 3; ++kind) o.res.live[kind] = 0;
}

// R4 + DESIGN §3 "locate": primary p gets id = words 0,1 of
// Philox(ctr = (p_lo, p_hi, 0, 0x5052494D), key = (seed_lo, seed_hi)).
int inject_one(Oracle &o, const Primary &p) {
  if (p.kind > 2u) return -1;
  const float depth = (float)o.geo.n_layers * o.pitch;
  if (!(p.pos[2] >= 0.0f) || !(p.pos[2] <= depth)) return -1;
  if (!(fabsf(p.pos[0]) <= o.geo.half_xy_mm) || !(fabsf(p.pos[1]) <= o.geo.half_xy_mm)) return -1;
  if (!(p.ekin >= o.tab.e_cut) || !(p.ekin <= o.tab.e_max)) return -1;
  Track t;
  for (int i = 0; i < 3; ++i) { t.pos[i] = p.pos[i]; t.dir[i] = p.dir[i]; t.nial[i] = -1.0f; }
  t.ekin = p.ekin;
  int layer = (int)(p.pos[2] / o.pitch);
  if (layer > (int)o.geo.n_layers - 1) layer = (int)o.geo.n_layers - 1;
  const float rel = p.pos[2] - (float)layer * o.pitch;
  t.vol = 2u * (uint32_t)layer + ((rel >= o.geo.abs_mm) ? 1u : 0u);
  const uint64_t idx = o.next_primary++;
  const uint32_t ctr[4] = {(uint32_t)idx, (uint32_t)(idx >> 32), 0u, 0x5052494Du};
  const uint32_t key[2] = {(uint32_t)o.seed, (uint32_t)(o.seed >> 32)};
  uint32_t w[4];
  philox4x32_10(ctr, key, w);
  t.id_lo = w[0];
  t.id_hi = w[1];
  t.step = 0;
  o.cur[p.kind].push_back(t);
  o.res.e_injected += (double)p.ekin + ((p.kind == KIND_EP) ? (double)o.two_mc2 : 0.0);
  o.res.live[p.kind] = o.cur[p.kind].size();
  if (o.cur[p.kind].size() > o.res.slots_used[p.kind]) o.res.slots_used[p.kind] = o.cur[p.kind].size();
  return 0;
}

bool any_live(const Oracle &o) {
  return !o.cur[0].empty() || !o.cur[1].empty() || !o.cur[2].empty();
}

}  // namespace

// ============================ C interface (ctypes) ==========================
extern "C" {

typedef struct orc_ctx orc_ctx;

void orc_philox4x32_10(const uint32_t *ctr, const uint32_t *key, uint32_t *out) {
  philox4x32_10(ctr, key, out);
}
void orc_philox_array(const uint32_t *ctr, const uint32_t *key, uint32_t *out, uint64_t n) {
  for (uint64_t i = 0; i < n; ++i) philox4x32_10(ctr + 4 * i, key + 2 * i, out + 4 * i);
}
void orc_u01_array(const uint32_t *x, float *out, uint64_t n) {
  for (uint64_t i = 0; i < n; ++i) out[i] = u01(x[i]);
}
void orc_lg_array(const float *x, float *out, uint64_t n) {
  for (uint64_t i = 0; i < n; ++i) out[i] = lg(x[i]);
}
void orc_ex_array(const float *x, float *out, uint64_t n) {
  for (uint64_t i = 0; i < n; ++i) out[i] = ex(x[i]);
}
void orc_sincos2pi_array(const float *u, float *sn, float *cs, uint64_t n) {
  for (uint64_t i = 0; i < n; ++i) sincos2pi(u[i], &sn[i], &cs[i]);
}
void orc_rotate_array(const float *d, const float *st, const float *ct, const float *sphi,
                      const float *cphi, float *out, uint64_t n) {
  for (uint64_t i = 0; i < n; ++i) rotate(d + 3 * i, st[i], ct[i], sphi[i], cphi[i], out + 3 * i);
}
// value of table (mat, group, qty) at kinetic energy E[i] (lnE = lg(E), rule T13)
void orc_lookup_array(const TablesIn *tin, uint32_t mat, uint32_t group, uint32_t qty,
                      const float *E, float *out, uint64_t n) {
  Tables t;
  t.n_bins = tin->n_bins; t.n_materials = tin->n_materials;
  t.e_min = tin->e_min; t.e_max = tin->e_max; t.ln_e_min = tin->ln_e_min;
  t.inv_dln = tin->inv_dln; t.e_cut = tin->e_cut;
  t.data.assign(tin->data, tin->data + (size_t)tin->n_materials * 6 * (tin->n_bins + 1));
  for (uint64_t i = 0; i < n; ++i) out[i] = interp(t.q(mat, (int)group, (int)qty), locate_bin(t, lg(E[i])));
}

orc_ctx *orc_create(const Geometry *g, const TablesIn *tin, uint64_t seed) {
  if (!g || !tin || !tin->data || g->n_layers == 0 || tin->n_bins == 0) return nullptr;
  if (g->mat_abs >= tin->n_materials || g->mat_gap >= tin->n_materials) return nullptr;
  Oracle *o = new Oracle();
  o->geo = *g;
  o->tab.n_bins = tin->n_bins; o->tab.n_materials = tin->n_materials;
  o->tab.e_min = tin->e_min; o->tab.e_max = tin->e_max; o->tab.ln_e_min = tin->ln_e_min;
  o->tab.inv_dln = tin->inv_dln; o->tab.e_cut = tin->e_cut;
  o->tab.data.assign(tin->data, tin->data + (size_t)tin->n_materials * 6 * (tin->n_bins + 1));
  o->tab.physics = tin->physics;
  if (tin->physics > 2u || (tin->physics >= 1u && !tin->data_x)) { delete o; return nullptr; }
  if (tin->physics >= 1u) o->tab.data_x.assign(tin->data_x, tin->data_x + (size_t)tin->n_materials * 3 * (tin->n_bins + 1));
  o->seed = seed;
  o->pitch = g->abs_mm + g->gap_mm;
  o->two_mc2 = 2.0f * o->mc2;
  o->edep.assign(2 * (size_t)g->n_layers, 0.0);
  return reinterpret_cast<orc_ctx *>(o);
}

void orc_destroy(orc_ctx *c) { delete reinterpret_cast<Oracle *>(c); }

// Primaries are injected immediately (batch = 0 semantics); see orc_run_batched.
int orc_inject(orc_ctx *c, const Primary *p, uint64_t n) {
  Oracle &o = *reinterpret_cast<Oracle *>(c);
  for (uint64_t i = 0; i < n; ++i)
    if (inject_one(o, p[i]) != 0) return -1;
  return 0;
}

// Queue primaries; orc_run_batched injects them `batch` at a time.
int orc_queue(orc_ctx *c, const Primary *p, uint64_t n) {
  Oracle &o = *reinterpret_cast<Oracle *>(c);
  o.pending.insert(o.pending.end(), p, p + n);
  return 0;
}

int orc_load_tracks(orc_ctx *c, uint32_t kind, const Track *t, uint64_t n) {
  if (kind > 2u) return -1;
  Oracle &o = *reinterpret_cast<Oracle *>(c);
  o.cur[kind].insert(o.cur[kind].end(), t, t + n);
  o.res.live[kind] = o.cur[kind].size();
  if (o.cur[kind].size() > o.res.slots_used[kind]) o.res.slots_used[kind] = o.cur[kind].size();
  return 0;
}

uint64_t orc_live(const orc_ctx *c, uint32_t kind) {
  return reinterpret_cast<const Oracle *>(c)->cur[kind].size();
}

int orc_read_tracks(const orc_ctx *c, uint32_t kind, Track *out, uint64_t cap, uint64_t *n) {
  const Oracle &o = *reinterpret_cast<const Oracle *>(c);
  const uint64_t m = o.cur[kind].size();
  *n = m;
  if (m > cap) return -2;
  if (m) std::memcpy(out, o.cur[kind].data(), m * sizeof(Track));
  return 0;
}

int orc_step(orc_ctx *c) {
  iterate(*reinterpret_cast<Oracle *>(c));
  return 0;
}

// Iterate until every buffer is empty (or max_iterations, 0 = unlimited).
int orc_run(orc_ctx *c, uint64_t max_iterations, int depth_first) {
  Oracle &o = *reinterpret_cast<Oracle *>(c);
  if (depth_first) { run_depth_first(o); return 0; }
  uint64_t it = 0;
  while (any_live(o) && (max_iterations == 0 || it < max_iterations)) { iterate(o); ++it; }
  return 0;
}

// PAPER.md:131 "-particles 25 -batch 5": each batch runs to extinction first.
int orc_run_batched(orc_ctx *c, uint64_t batch) {
  Oracle &o = *reinterpret_cast<Oracle *>(c);
  size_t done = 0;
  if (batch == 0) batch = o.pending.size();
  while (done < o.pending.size()) {
    const size_t hi = (done + batch < o.pending.size()) ? done + batch : o.pending.size();
    for (size_t i = done; i < hi; ++i)
      if (inject_one(o, o.pending[i]) != 0) return -1;
    done = hi;
    while (any_live(o)) iterate(o);
  }
  o.pending.clear();
  return 0;
}

void orc_get_result(const orc_ctx *c, Result *out, double *edep_slab) {
  const Oracle &o = *reinterpret_cast<const Oracle *>(c);
  *out = o.res;
  if (edep_slab) std::memcpy(edep_slab, o.edep.data(), o.edep.size() * sizeof(double));
}

// Rule R4: ids of primaries come from a running global index; a caller that simulates only a
// slice [lo, hi) of a larger primary list sets the index to lo first, so that every primary keeps
// the id (hence the random stream) it has in the unsliced run (sharding by event).
void orc_set_primary_index(orc_ctx *c, uint64_t next_index) {
  reinterpret_cast<Oracle *>(c)->next_primary = next_index;
}

void orc_reset_tallies(orc_ctx *c) {
  Oracle &o = *reinterpret_cast<Oracle *>(c);
  const uint64_t live[3] = {o.cur[0].size(), o.cur[1].size(), o.cur[2].size()};
  o.res = Result{};
  for (int k = 0; k < 3; ++k) { o.res.live[k] = live[k]; o.res.slots_used[k] = live[k]; }
  std::fill(o.edep.begin(), o.edep.end(), 0.0);
}

void orc_set_trace(orc_ctx *c, int on) {
  Oracle &o = *reinterpret_cast<Oracle *>(c);
  o.tracing = on != 0;
  o.trace.clear();
}
uint64_t orc_trace_size(const orc_ctx *c) { return reinterpret_cast<const Oracle *>(c)->trace.size(); }
void orc_read_trace(const orc_ctx *c, TraceRec *out) {
  const Oracle &o = *reinterpret_cast<const Oracle *>(c);
  if (!o.trace.empty()) std::memcpy(out, o.trace.data(), o.trace.size() * sizeof(TraceRec));
}

}  // extern "C"
