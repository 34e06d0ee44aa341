"""Pins for the table lookup (rule T13) and for the analytic table generator
(rules T12, T14, T15): closed forms, limits and an independent numerical
integration.  CPU only."""
import math

import numpy as np
from scipy import integrate

from oracle import math_fns
from workloads.tables import (ALPHA, GROUP_ELEC, GROUP_GAMMA, MATERIALS, MC2, Q_BREMS, Q_COMPT,
                              Q_PAIR, Q_PHOTO, Q_RANGE, Q_STOP, R_E, SIGMA_THOMSON, build_tables,
                              constant_tables, klein_nishina_per_electron, stopping_power)

E_CUT = 0.1


def test_lookup_reproduces_ln_linear_tables_and_nodes():
    tab = constant_tables(64, E_CUT, 100.0, E_CUT)
    a, b = 0.7, 0.31
    tab.data[0, GROUP_GAMMA, Q_COMPT] = (a + b * np.log(tab.nodes)).astype(np.float32)
    rng = np.random.default_rng(1)
    E = np.exp(rng.uniform(math.log(E_CUT), math.log(100.0), 50000)).astype(np.float32)
    v = math_fns.lookup(tab, 0, GROUP_GAMMA, Q_COMPT, E)
    ref = a + b * np.log(E.astype(np.float64))
    assert np.abs(v - ref).max() < 3e-6
    # other quantities/materials are not mixed in (index arithmetic of rule T14)
    tab.data[1, GROUP_ELEC, Q_RANGE] = 7.0
    assert (math_fns.lookup(tab, 1, GROUP_ELEC, Q_RANGE, E[:100]) == 7.0).all()
    assert (math_fns.lookup(tab, 1, GROUP_ELEC, Q_STOP, E[:100]) == 0.0).all()
    # nodes reproduce, end points included (primaries sit exactly on the last node)
    real = build_tables(64, E_CUT, 100.0, E_CUT)
    nodes = real.nodes.astype(np.float32)
    for (g, q) in ((GROUP_GAMMA, Q_COMPT), (GROUP_ELEC, Q_RANGE), (GROUP_ELEC, Q_STOP)):
        v = math_fns.lookup(real, 0, g, q, nodes)
        assert np.allclose(v, real.data[0, g, q], rtol=2e-5)
    v_end = math_fns.lookup(real, 0, GROUP_ELEC, Q_RANGE, np.float32([100.0]))[0]
    assert abs(v_end / real.data[0, GROUP_ELEC, Q_RANGE, -1] - 1) < 2e-5


def test_grid_definition():
    t = build_tables(256, E_CUT, 1.0e4, E_CUT)
    assert t.data.shape == (2, 2, 3, 257) and t.data.dtype == np.float32
    assert t.nodes[0] == E_CUT and t.nodes[-1] == 1.0e4
    assert np.allclose(np.diff(np.log(t.nodes)), math.log(1e5) / 256, rtol=1e-12)
    assert t.inv_dln == np.float32(256 / math.log(1e5)) and t.ln_e_min == np.float32(math.log(0.1))


def test_klein_nishina_against_numerical_integration_and_thomson_limit():
    def dsigma(ct, k):
        r = 1.0 / (1.0 + k * (1.0 - ct))
        return math.pi * R_E * R_E * r * r * (r + 1.0 / r - (1.0 - ct * ct))   # 2 pi sin(t) dt folded in
    for E in (0.1, 1.0, 10.0, 1000.0):
        k = E / MC2
        num, _ = integrate.quad(dsigma, -1.0, 1.0, args=(k,), epsabs=0, epsrel=1e-10)
        assert abs(klein_nishina_per_electron(E) / num - 1) < 1e-8
    assert abs(klein_nishina_per_electron(1e-5) / SIGMA_THOMSON - 1) < 1e-4


def test_pair_photo_brems_stopping_closed_forms():
    pb, lar = MATERIALS
    t = build_tables(256, E_CUT, 1.0e4, E_CUT)
    pair = t.data[0, GROUP_GAMMA, Q_PAIR].astype(np.float64)
    assert (pair[t.nodes <= 2 * MC2] == 0).all() and (np.diff(pair) >= 0).all()
    assert abs(pair[-1] - 7.0 / (9.0 * pb.X0)) < 1e-6                  # complete-screening asymptote
    photo = t.data[0, GROUP_GAMMA, Q_PHOTO].astype(np.float64)
    slope = np.diff(np.log(photo)) / np.diff(np.log(t.nodes))
    assert np.allclose(slope, -3.5, atol=1e-4)                          # ~ Z^5 / E^3.5
    ratio = t.data[0, GROUP_GAMMA, Q_PHOTO, 0] / t.data[1, GROUP_GAMMA, Q_PHOTO, 0]
    assert abs(ratio / ((pb.n_atoms * pb.Z**5) / (lar.n_atoms * lar.Z**5)) - 1) < 1e-6
    # mean radiative loss: int_cut^T k dSigma/dk dk + cut/X0 * ... = T/X0  (rule T15)
    brems = t.data[0, GROUP_ELEC, Q_BREMS].astype(np.float64)
    assert np.allclose(brems, np.log(t.nodes / E_CUT) / pb.X0, rtol=1e-6, atol=1e-9)
    # minimum-ionising stopping power of Pb ~ 1.1-1.3 MeV cm^2/g (PDG-scale sanity, not parity-critical)
    col = stopping_power(pb, t.nodes, E_CUT) - E_CUT / pb.X0
    assert 1.0 < col.min() / (pb.rho * 0.1) < 1.4
    # dR/dT = 1/S
    R = t.data[0, GROUP_ELEC, Q_RANGE].astype(np.float64)
    S = t.data[0, GROUP_ELEC, Q_STOP].astype(np.float64)
    mid = slice(1, -1)
    dRdT = (R[2:] - R[:-2]) / (t.nodes[2:] - t.nodes[:-2])
    assert np.allclose(dRdT, 1.0 / S[mid], rtol=5e-3)
    assert abs(R[0] - E_CUT / S[0]) < 1e-6
