// One transport step of one track (DESIGN.md rules S16-S27, S31).
//
// The paper's per-type kernels read a track, ask the physics library for the step
// length from the numbers of interaction lengths left (Fig. 3, "NumIALeft"), ask the
// geometry for the distance to the next boundary, move, apply continuous loss and the discrete
// interaction, and initialise secondaries from the parent's position and navigation state (Fig. 2,
// PAPER.md:47-60).  The physics itself is BASELINE.json's simplified analytic model; every formula
// below is the rule of DESIGN.md §3 named in its comment, in that rule's operation order (the order
// is part of the rule: rule M7 makes results bit-reproducible).
//
// Everything lives in registers; the only memory touched is the shared-memory copy of the tables.
#pragma once
#include <cstdint>
#include <cuda_runtime.h>

#include "layout.cuh"
#include "mathfn.cuh"
#include "rng.cuh"

namespace adept {

enum Kind : int { K_EM = 0, K_EP = 1, K_GAMMA = 2 };

// What the step needs besides the track: tables (shared memory) and geometry (registers).
struct Env {
  const float4 *tab;  // the particle group's tables: [material][node] -> {qty0, qty1, qty2, qty3 or 0}
  uint32_t group_nodes;  // nodes of one staged group (materials * nodes): the e+ extras follow the e+- group
  uint32_t nodes;     // n_bins + 1
  float ln_e_min, inv_dln, e_cut;
  uint32_t n_slabs;   // 2 * n_layers
  float abs_mm, pitch, half_xy;
  uint32_t mat_abs, mat_gap;
};

struct Kid {  // a secondary: position, slab, nial = -1, step = 0 come from the parent (S28, R6)
  float dx, dy, dz, ekin;
  uint32_t id_lo, id_hi;
  int kind;  // -1 = none
};

// The step is split in two so that a warp never drags idle lanes through an interaction:
//   move_*      rules S17(test)-S25: everything up to and including the boundary crossing.  Most
//               tracks end their step here.  A track whose step ends in a discrete interaction
//               (or an e+ that must annihilate) is only *marked* (MoveOut::pending).
//   interact_*  rule S26 (and the S17 annihilation): run later by the kernel on a dense batch of
//               marked tracks, so that the Philox blocks of calls 1 and 2 and the sampling code are
//               executed by full warps.
// Both halves together are exactly the rule sequence; the split changes no operation and no operand.
enum Pending : int { P_NONE = -1, P_PROC0 = 0, P_PROC1 = 1, P_PROC2 = 2, P_ANNIH = 4 };

// Energy tallies are sums of fp32 terms (rule M7); a step hands its terms over one by one:
// at most two deposits in the step's slab, and the track's whole energy when it escapes (S25) or
// trips the runaway guard (S31) -- the kernel adds them to its accumulators (step_impl.cuh).
struct MoveOut {
  bool alive;    // track goes to the next iteration (meaningless while pending)
  bool escaped;  // left the calorimeter (S25): ekin (+ 2 mc^2 for e+) is carried out
  bool guard;    // S31: ekin (+ 2 mc^2 for e+) is deposited in the post-step slab
  int pending;   // Pending: interaction still to be done
  float dep;     // energy deposited in the pre-step slab (0 = none)
  float dep_b;   // second term into the same slab (0 = none)
};

struct InteractOut {
  bool alive;
  bool guard;   // S31
  Kid kid[2];   // by child ordinal (R5)
  float dep;    // deposited in the track's slab (interactions do not change slab)
  float dep_b;  // second term into the same slab
};

constexpr float kInf = __builtin_huge_valf();
constexpr float kMc2 = 0.51099895f;
__device__ __forceinline__ float two_mc2() { return 2.0f * kMc2; }

// T13: position on the log grid
struct Bin {
  int j;
  float f;
};
__device__ __forceinline__ Bin locate_bin(const Env &g, float lnE) {
  const float x = (lnE - g.ln_e_min) * g.inv_dln;
  int j = static_cast<int>(x);
  const int last = static_cast<int>(g.nodes) - 2;
  j = j < 0 ? 0 : j;
  j = j > last ? last : j;
  Bin b;
  b.j = j;
  b.f = x - static_cast<float>(j);
  return b;
}
__device__ __forceinline__ float lerp_node(float f, float lo, float hi) { return fmaf(f, hi - lo, lo); }

// S21 geometry of slab i
__device__ __forceinline__ float slab_zlo(const Env &g, uint32_t i) {
  return fmaf(static_cast<float>(i >> 1), g.pitch, (i & 1u) ? g.abs_mm : 0.0f);
}

enum Face : int { FACE_ZP = 0, FACE_ZM = 1, FACE_XY = 2 };

// The rule's `valid ? n / d : +inf`.  The divisor is selected first (1 where the quotient is not
// used), so that no lane divides by zero: a zero divisor sends the whole warp through the slow path
// of the IEEE division (Sigma_pair is exactly 0 below ~3.4 MeV, i.e. for a third of the photons).
// The empty asm keeps the compiler from undoing the selection (it otherwise proves the quotient
// unused on those lanes and divides by the raw value).
__device__ __forceinline__ float quotient_or_inf(float n, float d, bool valid) {
  float dd = valid ? d : 1.0f;
  asm("" : "+f"(dd));
  const float q = n / dd;
  return valid ? q : kInf;
}

// S21: distance to the slab faces and the transverse box, and which face is hit first.
__device__ __forceinline__ float geometry_step(const Trk &t, const Env &g, float z_lo, float z_hi, int &face) {
  const float H = g.half_xy;
  // each quotient is the rule's (plane - pos) / dir; the plane is selected first so that a warp
  // executes one division per axis whatever the signs of its lanes' directions
  const float n_z = ((t.dz > 0.0f) ? z_hi : z_lo) - t.pz;
  const float n_x = ((t.dx > 0.0f) ? H : -H) - t.px;
  const float n_y = ((t.dy > 0.0f) ? H : -H) - t.py;
  const float s_z = quotient_or_inf(n_z, t.dz, t.dz != 0.0f);
  const float s_x = quotient_or_inf(n_x, t.dx, t.dx != 0.0f);
  const float s_y = quotient_or_inf(n_y, t.dy, t.dy != 0.0f);
  float s_g = s_z;
  face = (t.dz > 0.0f) ? FACE_ZP : FACE_ZM;
  if (s_x < s_g) { s_g = s_x; face = FACE_XY; }
  if (s_y < s_g) { s_g = s_y; face = FACE_XY; }
  if (!(s_g > 0.0f)) s_g = 0.0f;
  return s_g;
}

// S25, applied where `doit` holds: snap to the plane and change slab, or escape.  Returns true if the
// track escaped.  Written with selects throughout: the faces (and whether the step ends on a face
// at all) differ between the lanes of a warp, a branch per case would serialise them.
__device__ __forceinline__ bool cross_boundary(bool doit, Trk &t, const Env &g, uint32_t vol0, int face, float z_lo,
                                               float z_hi) {
  const bool zp = face == FACE_ZP, zm = face == FACE_ZM;
  const uint32_t vol_new = zp ? vol0 + 1u : vol0 - 1u;  // vol0 - 1 wraps for slab 0: caught by the range test
  const bool out = (face == FACE_XY) || (vol_new >= g.n_slabs);
  const float pz_new = zp ? z_hi : (zm ? z_lo : t.pz);
  t.pz = doit ? pz_new : t.pz;
  t.vol = (doit && !out) ? vol_new : vol0;
  return doit && out;
}

__device__ __forceinline__ void make_kid(Kid &k, int kind, float dx, float dy, float dz, float ekin, uint32_t id_lo,
                                         uint32_t id_hi) {
  k.kind = kind; k.dx = dx; k.dy = dy; k.dz = dz; k.ekin = ekin; k.id_lo = id_lo; k.id_hi = id_hi;
}

// S27: rotate unit vector d by polar (st, ct) and azimuth (sphi, cphi); renormalise.
__device__ __forceinline__ void rotate_dir(float dx, float dy, float dz, float st, float ct, float sphi, float cphi,
                                           float &ox, float &oy, float &oz) {
  const float q2 = fmaf(-dz, dz, 1.0f);
  float a, b, c;
  if (q2 > 1e-10f) {
    const float sp = sqrtf(q2);
    const float ux = ((dx * dz) * cphi - dy * sphi) / sp;
    const float uy = ((dy * dz) * cphi + dx * sphi) / sp;
    const float uz = -(sp * cphi);
    a = fmaf(st, ux, ct * dx);
    b = fmaf(st, uy, ct * dy);
    c = fmaf(st, uz, ct * dz);
  } else {
    a = st * cphi;
    b = st * sphi;
    c = (dz < 0.0f) ? -ct : ct;
  }
  const float nn = sqrtf(fmaf(a, a, fmaf(b, b, c * c)));
  ox = a / nn;
  oy = b / nn;
  oz = c / nn;
}

__device__ __forceinline__ void move_out_init(MoveOut &o) {
  o.alive = true; o.escaped = false; o.guard = false; o.pending = P_NONE; o.dep = 0.0f; o.dep_b = 0.0f;
}
__device__ __forceinline__ void interact_out_init(InteractOut &o) {
  o.alive = true; o.guard = false; o.kid[0].kind = -1; o.kid[1].kind = -1; o.dep = 0.0f; o.dep_b = 0.0f;
}

// S31: runaway guard
template <int KIND, typename Out> __device__ __forceinline__ void runaway_guard(Trk &t, Out &o) {
  if (t.step >= (1u << 20)) {
    o.guard = true;
    o.alive = false;
  }
}

// ------------------------------------------------------------------------------ photon -------
__device__ __forceinline__ void move_gamma(Trk &t, const Env &g, MoveOut &o) {
  move_out_init(o);
  const Stream rs{t.id_lo, t.id_hi, t.step};

  // S18: re-sample spent interaction lengths (pair, Compton, photoelectric)
  if (t.n0 <= 0.0f || t.n1 <= 0.0f || t.n2 <= 0.0f) {
    const uint4 r = rs.call(0);
    if (t.n0 <= 0.0f) t.n0 = -lg(u01(r.x));
    if (t.n1 <= 0.0f) t.n1 = -lg(u01(r.y));
    if (t.n2 <= 0.0f) t.n2 = -lg(u01(r.z));
  }

  // S19: cross sections at the pre-step energy and material
  const uint32_t vol0 = t.vol;
  const uint32_t mat = (vol0 & 1u) ? g.mat_gap : g.mat_abs;
  const Bin b = locate_bin(g, lg(t.ekin));
  const float4 *node = g.tab + mat * g.nodes + b.j;
  const float4 A = node[0], B = node[1];
  const float sig0 = lerp_node(b.f, A.x, B.x);
  const float sig1 = lerp_node(b.f, A.y, B.y);
  const float sig2 = lerp_node(b.f, A.z, B.z);
  // s_j = nial_j / Sigma_j where Sigma_j > 0, else +inf
  const float s0 = quotient_or_inf(t.n0, sig0, sig0 > 0.0f);
  const float s1 = quotient_or_inf(t.n1, sig1, sig1 > 0.0f);
  const float s2 = quotient_or_inf(t.n2, sig2, sig2 > 0.0f);

  // S21
  const float z_lo = slab_zlo(g, vol0), z_hi = slab_zlo(g, vol0 + 1u);
  int face;
  float s = geometry_step(t, g, z_lo, z_hi, face);

  // S22: strict '<', earlier candidate wins ties
  int w = -1;
  if (s0 < s) { s = s0; w = 0; }
  if (s1 < s) { s = s1; w = 1; }
  if (s2 < s) { s = s2; w = 2; }

  // S23
  t.px = fmaf(s, t.dx, t.px);
  t.py = fmaf(s, t.dy, t.py);
  t.pz = fmaf(s, t.dz, t.pz);
  t.n0 = fmaf(-s, sig0, t.n0);
  t.n1 = fmaf(-s, sig1, t.n1);
  t.n2 = fmaf(-s, sig2, t.n2);
  t.step = rs.step + 1u;

  // what the step ends in, as flags (no early exits: the outcomes of a warp's lanes differ)
  const bool geom = w < 0;
  o.pending = geom ? int(P_NONE) : w;                              // S26 follows in interact_gamma
  o.escaped = cross_boundary(geom, t, g, vol0, face, z_lo, z_hi);  // S25
  o.guard = geom && !o.escaped && t.step >= (1u << 20);            // S31
  o.alive = !(o.escaped || o.guard);
}

// S26 for a photon whose step (already taken: t.step is the post-increment value) ended in process w.
// PHYS = 1: the Compton energy fraction comes from the full Klein-Nishina distribution (rule X37).
template <int PHYS> __device__ __forceinline__ void interact_gamma(Trk &t, int w, const Env &g, InteractOut &o) {
  interact_out_init(o);
  const Stream rs{t.id_lo, t.id_hi, t.step - 1u};  // draws are addressed by the pre-increment step (R2)
  const uint4 r1 = rs.call(1), r2 = rs.call(2);
  if (w == 0) {  // pair: uniform split of E - 2 mc^2, both along dir; photon dies
    const float E_av = t.ekin - two_mc2();
    const float T_minus = u01(r1.x) * E_av;
    const float T_plus = E_av - T_minus;
    if (T_minus >= g.e_cut) make_kid(o.kid[0], K_EM, t.dx, t.dy, t.dz, T_minus, r2.x, r2.y);
    else o.dep = T_minus;
    make_kid(o.kid[1], K_EP, t.dx, t.dy, t.dz, T_plus, r2.z, r2.w);
    o.alive = false;
    return;
  }
  if (w == 2) {  // photoelectric: e- with T = E along dir; photon dies
    make_kid(o.kid[0], K_EM, t.dx, t.dy, t.dz, t.ekin, r2.x, r2.y);
    o.alive = false;
    return;
  }
  // Compton: 1/eps spectrum on [1/(1+2 kappa), 1], exact kinematics
  t.n1 = -1.0f;
  const float E = t.ekin;
  const float kappa = E / kMc2;
  const float L = lg(fmaf(2.0f, kappa, 1.0f));
  float eps;
  if constexpr (PHYS == 0) {
    eps = ex(-(u01(r1.x) * L));
  } else {
    // X37: composition (1/eps on [eps0, 1] with weight a1, eps on [eps0, 1] with weight a2) and
    // rejection by g = 1 - eps sin^2(theta) / (1 + eps^2); try k draws call 3 + k, at most 16 tries
    const float eps0 = 1.0f / fmaf(2.0f, kappa, 1.0f);
    const float eps0sq = eps0 * eps0;
    const float a1 = L;
    const float a2 = 0.5f * (1.0f - eps0sq);
    const float thr = a1 / (a1 + a2);
    eps = 1.0f;
    for (int k = 0; k < 16; ++k) {
      const uint4 r = rs.call(3u + uint32_t(k));
      const float u1 = u01(r.x), u2 = u01(r.y), u3 = u01(r.z);
      if (thr > u1) eps = ex(-(a1 * u2));
      else eps = sqrtf(fmaf(1.0f - eps0sq, u2, eps0sq));
      if (eps < eps0) eps = eps0;
      if (eps > 1.0f) eps = 1.0f;
      const float tt = (1.0f - eps) / (kappa * eps);
      const float sin2 = tt * (2.0f - tt);
      const float gg = 1.0f - (eps * sin2) / fmaf(eps, eps, 1.0f);
      if (gg >= u3) break;
    }
  }
  const float E1 = eps * E;
  const float T = E - E1;
  float ct = 1.0f - (((1.0f / eps) - 1.0f) / kappa);
  if (ct > 1.0f) ct = 1.0f;
  if (ct < -1.0f) ct = -1.0f;
  const float st = sqrtf(fmaf(-ct, ct, 1.0f));
  float sphi, cphi;
  sincos2pi(u01(r1.y), sphi, cphi);
  float nx, ny, nz;
  rotate_dir(t.dx, t.dy, t.dz, st, ct, sphi, cphi, nx, ny, nz);
  const float qx = fmaf(E, t.dx, -(E1 * nx));
  const float qy = fmaf(E, t.dy, -(E1 * ny));
  const float qz = fmaf(E, t.dz, -(E1 * nz));
  const float pn = sqrtf(fmaf(qx, qx, fmaf(qy, qy, qz * qz)));
  if (T >= g.e_cut && pn > 0.0f) make_kid(o.kid[0], K_EM, qx / pn, qy / pn, qz / pn, T, r2.x, r2.y);
  else o.dep = T;
  if (E1 < g.e_cut) {
    o.dep_b = E1;
    o.alive = false;
    return;
  }
  t.ekin = E1;
  t.dx = nx; t.dy = ny; t.dz = nz;
  runaway_guard<K_GAMMA>(t, o);
}

// --------------------------------------------------------------------- electron / positron ---
// PHYS = 1: delta-ray production is a second discrete process, on nial[1] (rule X36).
// PHYS = 2: also multiple scattering (rule X39): a third step limiter and a deflection after the move.
template <int KIND, int PHYS> __device__ __forceinline__ void move_elec(Trk &t, const Env &g, MoveOut &o) {
  constexpr bool MSC = PHYS == 2;
  static_assert(KIND == K_EM || KIND == K_EP, "e- or e+");
  move_out_init(o);
  const Stream rs{t.id_lo, t.id_hi, t.step};
  const float e_cut = g.e_cut;

  // S17: a positron below the cut annihilates at rest, first (done in interact_elec; the track is
  // untouched here, in particular its step counter)
  if (KIND == K_EP && t.ekin < e_cut) {
    o.pending = P_ANNIH;
    return;
  }

  // S18: bremsstrahlung is the only discrete process; nial[1], nial[2] are carried unchanged
  // (X36: delta-ray production is the second one, nial[2] is carried unchanged)
  if constexpr (PHYS == 0) {
    if (t.n0 <= 0.0f) t.n0 = -lg(u01(rs.call(0).x));
  } else {
    if (t.n0 <= 0.0f || t.n1 <= 0.0f || (KIND == K_EP && t.n2 <= 0.0f)) {
      const uint4 r = rs.call(0);
      if (t.n0 <= 0.0f) t.n0 = -lg(u01(r.x));
      if (t.n1 <= 0.0f) t.n1 = -lg(u01(r.y));
      if (KIND == K_EP && t.n2 <= 0.0f) t.n2 = -lg(u01(r.z));
    }
  }

  // S19, S20
  const uint32_t vol0 = t.vol;
  const uint32_t mat = (vol0 & 1u) ? g.mat_gap : g.mat_abs;
  const float E0 = t.ekin;
  const Bin b = locate_bin(g, lg(E0));
  const float4 *tab = g.tab + mat * g.nodes;
  const float4 A = tab[b.j], B = tab[b.j + 1];
  const float sig0 = lerp_node(b.f, A.x, B.x);
  const float S0 = lerp_node(b.f, A.y, B.y);
  const float R = lerp_node(b.f, A.z, B.z);
  const float s0 = quotient_or_inf(t.n0, sig0, sig0 > 0.0f);
  float sig1 = 0.0f, s1 = kInf, sig2 = 0.0f, s2 = kInf;
  if constexpr (PHYS != 0) {
    sig1 = lerp_node(b.f, A.w, B.w);  // X36: Sigma_delta rides in the fourth lane of the e+- group
    s1 = quotient_or_inf(t.n1, sig1, sig1 > 0.0f);
    if constexpr (KIND == K_EP) {     // X38: Sigma_annihilation, first lane of the e+ extras staged behind the group
      const float4 *tx = tab + g.group_nodes;
      sig2 = lerp_node(b.f, tx[b.j].x, tx[b.j + 1].x);
      s2 = quotient_or_inf(t.n2, sig2, sig2 > 0.0f);
    }
  }
  float s_e;
  {
    const float r_min = 0.1f, f_r = 0.2f;
    const float fr = f_r * R;
    s_e = (R <= r_min) ? R : ((fr > r_min) ? fr : r_min);
  }

  // S21
  const float z_lo = slab_zlo(g, vol0), z_hi = slab_zlo(g, vol0 + 1u);
  int face;
  float s = geometry_step(t, g, z_lo, z_hi, face);

  // X39a, X39b: multiple-scattering limit max(DynamicRangeFactor * InitialRange, TlimitMin); the three
  // words are (re-)initialised at the start of a track and after a slab crossing (InitialRange < 0)
  float sig_tr = 0.0f, s_m = kInf;
  if constexpr (MSC) {
    const float4 *tx = tab + g.group_nodes;
    sig_tr = lerp_node(b.f, tx[b.j].y, tx[b.j + 1].y);
    if (sig_tr > 0.0f) {
      if (t.m0 < 0.0f) {
        float safety = fminf(t.pz - z_lo, z_hi - t.pz);
        if (!(safety > 0.0f)) safety = 0.0f;
        t.m0 = R;
        t.m1 = fmaxf(0.04f, (0.6f * safety) / R);
        t.m2 = fmaxf(1e-3f, 0.01f / sig_tr);
      }
      s_m = fmaxf(t.m1 * t.m0, t.m2);
    }
  }

  // S22: GEOM (-1), ELOSS (3), multiple scattering (5), brems (0), delta (1), annihilation in flight (2)
  int w = -1;
  if (s_e < s) { s = s_e; w = 3; }
  if (MSC && s_m < s) { s = s_m; w = 5; }
  if (s0 < s) { s = s0; w = 0; }
  if (PHYS != 0 && s1 < s) { s = s1; w = 1; }
  if (PHYS != 0 && KIND == K_EP && s2 < s) { s = s2; w = 2; }

  // S23
  t.px = fmaf(s, t.dx, t.px);
  t.py = fmaf(s, t.dy, t.py);
  t.pz = fmaf(s, t.dz, t.pz);
  t.n0 = fmaf(-s, sig0, t.n0);
  if constexpr (PHYS != 0) t.n1 = fmaf(-s, sig1, t.n1);
  if constexpr (PHYS != 0 && KIND == K_EP) t.n2 = fmaf(-s, sig2, t.n2);
  t.step = rs.step + 1u;

  // S24: continuous loss by the midpoint rule, deposit in the pre-step slab
  float E_post;
  {
    float E_mid = fmaf(-0.5f * s, S0, E0);
    if (!(E_mid > e_cut)) E_mid = e_cut;
    const Bin bm = locate_bin(g, lg(E_mid));
    const float S_mid = lerp_node(bm.f, tab[bm.j].y, tab[bm.j + 1].y);
    float dE = s * S_mid;
    if (!(dE < E0)) dE = E0;
    E_post = E0 - dE;
    if (w == 3 && s >= R) E_post = 0.0f;  // the track stops
  }
  o.dep = E0 - E_post;
  t.ekin = E_post;
  // what the step ends in, as flags (no early exits: the outcomes of a warp's lanes differ)
  const bool below = E_post < e_cut;            // S24: e- deposits the rest and dies; e+ is kept for S17
  if constexpr (MSC) {
    // X39c: deflection along the step, 1 - cos(theta) exponential with mean s Sigma_tr (draws of call 3)
    if (!below && sig_tr > 0.0f && s > 0.0f) {
      const uint4 r = rs.call(3);
      const float tau = s * sig_tr;
      float c = fmaf(tau, lg(u01(r.x)), 1.0f);
      if (c < -1.0f) c = -1.0f;
      const float sn = sqrtf(fmaf(-c, c, 1.0f));
      float sphi, cphi;
      sincos2pi(u01(r.y), sphi, cphi);
      float nx, ny, nz;
      rotate_dir(t.dx, t.dy, t.dz, sn, c, sphi, cphi, nx, ny, nz);
      t.dx = nx; t.dy = ny; t.dz = nz;
    }
  }
  const bool brems = !below && (w == 0 || w == 1 || w == 2);  // S26 (X36: w == 1, X38: w == 2) follows in interact_elec
  const bool geom = !below && w < 0;
  o.dep_b = (below && KIND == K_EM) ? E_post : 0.0f;
  o.pending = brems ? w : int(P_NONE);
  o.escaped = cross_boundary(geom, t, g, vol0, face, z_lo, z_hi);  // S25
  if (MSC && t.vol != vol0) t.m0 = -1.0f;                          // X39d: a new slab, a new InitialRange
  o.guard = !below && !brems && !o.escaped && t.step >= (1u << 20);  // S31
  o.alive = !((below && KIND == K_EM) || o.escaped || o.guard);
}

// S17 annihilation (pending == P_ANNIH: track untouched) or S26 bremsstrahlung (step already taken).
template <int KIND, int PHYS> __device__ __forceinline__ void interact_elec(Trk &t, int pending, const Env &g, InteractOut &o) {
  interact_out_init(o);
  const bool annih = (KIND == K_EP) && (pending == P_ANNIH);
  const Stream rs{t.id_lo, t.id_hi, annih ? t.step : t.step - 1u};
  const uint4 r1 = rs.call(1), r2 = rs.call(2);
  if (annih) {  // two back-to-back photons of energy mc^2, isotropic
    o.dep = t.ekin;
    const float ct = 1.0f - 2.0f * u01(r1.z);
    const float st = sqrtf(fmaf(-ct, ct, 1.0f));
    float sphi, cphi;
    sincos2pi(u01(r1.w), sphi, cphi);
    const float ax = st * cphi, ay = st * sphi, az = ct;
    make_kid(o.kid[0], K_GAMMA, ax, ay, az, kMc2, r2.x, r2.y);
    make_kid(o.kid[1], K_GAMMA, -ax, -ay, -az, kMc2, r2.z, r2.w);
    o.alive = false;
    return;
  }
  const float e_cut = g.e_cut;
  if (PHYS != 0 && KIND == K_EP && pending == P_PROC2) {
    // X38: annihilation in flight, two photons isotropic in the centre-of-momentum frame
    const float E = t.ekin;
    const float e_tot = E + two_mc2();
    const float pp = sqrtf(E * e_tot);
    const float beta = pp / e_tot;
    const float cs = 1.0f - 2.0f * u01(r1.z);
    const float k1 = (0.5f * e_tot) * fmaf(beta, cs, 1.0f);
    const float k2 = e_tot - k1;
    float c1 = (cs + beta) / fmaf(beta, cs, 1.0f);
    if (c1 > 1.0f) c1 = 1.0f;
    if (c1 < -1.0f) c1 = -1.0f;
    const float s1 = sqrtf(fmaf(-c1, c1, 1.0f));
    float sphi, cphi;
    sincos2pi(u01(r1.w), sphi, cphi);
    float ax, ay, az;
    rotate_dir(t.dx, t.dy, t.dz, s1, c1, sphi, cphi, ax, ay, az);
    const float qx = fmaf(pp, t.dx, -(k1 * ax));
    const float qy = fmaf(pp, t.dy, -(k1 * ay));
    const float qz = fmaf(pp, t.dz, -(k1 * az));
    const float qn = sqrtf(fmaf(qx, qx, fmaf(qy, qy, qz * qz)));
    if (k1 >= e_cut) make_kid(o.kid[0], K_GAMMA, ax, ay, az, k1, r2.x, r2.y);
    else o.dep = k1;
    if (k2 >= e_cut && qn > 0.0f) make_kid(o.kid[1], K_GAMMA, qx / qn, qy / qn, qz / qn, k2, r2.z, r2.w);
    else o.dep_b = k2;
    o.alive = false;
    return;
  }
  if (PHYS != 0 && pending == P_PROC1) {
    // X36: delta ray from the 1/T^2 spectrum on [e_cut, E/2], two-body kinematics on a free electron
    t.n1 = -1.0f;
    const float E = t.ekin;
    const float a = e_cut, b = 0.5f * E;
    if (!(b > a)) {   // guard of rule X36: post-step energy at or below 2 e_cut, no delta ray can be made
      runaway_guard<KIND>(t, o);
      return;
    }
    float T = (a * b) / (b - u01(r1.x) * (b - a));
    if (!(T > a)) T = a;
    if (!(T < b)) T = b;
    const float E1 = E - T;
    const float tau = E + two_mc2();
    float cd = sqrtf((T * tau) / (E * (T + two_mc2())));
    float cp = sqrtf((E1 * tau) / (E * (E1 + two_mc2())));
    if (cd > 1.0f) cd = 1.0f;
    if (cp > 1.0f) cp = 1.0f;
    const float sd = sqrtf(fmaf(-cd, cd, 1.0f));
    const float sp = sqrtf(fmaf(-cp, cp, 1.0f));
    float sphi, cphi;
    sincos2pi(u01(r1.y), sphi, cphi);
    float ax, ay, az, bx, by, bz;
    rotate_dir(t.dx, t.dy, t.dz, sd, cd, sphi, cphi, ax, ay, az);
    rotate_dir(t.dx, t.dy, t.dz, sp, cp, -sphi, -cphi, bx, by, bz);
    make_kid(o.kid[0], K_EM, ax, ay, az, T, r2.x, r2.y);
    t.ekin = E1;
    t.dx = bx; t.dy = by; t.dz = bz;
    runaway_guard<KIND>(t, o);
    return;
  }
  // bremsstrahlung: k from the 1/k spectrum on [e_cut, E], photon along dir
  t.n0 = -1.0f;
  const float E = t.ekin;
  float k = e_cut * ex(u01(r1.x) * lg(E / e_cut));
  if (!(k < E)) k = E;
  make_kid(o.kid[0], K_GAMMA, t.dx, t.dy, t.dz, k, r2.x, r2.y);
  const float E_new = E - k;
  if (E_new < e_cut && KIND == K_EM) {
    o.dep = E_new;
    o.alive = false;
    return;
  }
  t.ekin = E_new;
  runaway_guard<KIND>(t, o);
}

}  // namespace adept
