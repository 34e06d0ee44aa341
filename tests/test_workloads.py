"""The seeded input generators: pure functions of the seed, with the shapes and
distributions BASELINE.json's configs state.  They hold no transport arithmetic."""
import numpy as np

from workloads import CONFIGS, gen_primaries, gen_sweep, gen_tracks, geometry_for, tables_for


def test_single_step_population_matches_config_3():
    c = CONFIGS["single_step"]
    geo = geometry_for("single_step")
    n = 200_000
    a = gen_tracks(n, c["seed"], geo, c["e_max"], c["fractions"])
    b = gen_tracks(n, c["seed"], geo, c["e_max"], c["fractions"])
    assert all((x.tobytes() == y.tobytes()) for x, y in zip(a, b))                  # deterministic
    assert [p.shape[0] for p in a] == [80_000, 20_000, 100_000]                     # 40 / 10 / 50 %
    assert gen_tracks(n, c["seed"] + 1, geo, c["e_max"], c["fractions"])[0].tobytes() != a[0].tobytes()
    t = np.concatenate(a)
    depth = geo.n_layers * (geo.abs_mm + geo.gap_mm)
    assert (t["pos"][:, 2] >= 0).all() and (t["pos"][:, 2] <= depth).all()
    assert (np.abs(t["pos"][:, :2]) <= geo.half_xy_mm).all()
    assert np.allclose(np.linalg.norm(t["dir"].astype(np.float64), axis=1), 1.0, atol=1e-6)
    assert abs(t["dir"][:, 2].mean()) < 0.01                                        # isotropic
    assert (t["ekin"] >= 0.1).all() and (t["ekin"] <= c["e_max"]).all()
    le = np.log(t["ekin"].astype(np.float64))
    assert abs(le.mean() - 0.5 * (np.log(0.1) + np.log(c["e_max"]))) < 0.05         # log-uniform
    assert (t["nial"] > 0).all() and abs(t["nial"].mean() - 1.0) < 0.01             # exponential(1)
    assert (t["vol"] < 2 * geo.n_layers).all() and (t["step"] == 0).all()
    # the slab index is the slab that contains z
    pitch = geo.abs_mm + geo.gap_mm
    layer = np.minimum((t["pos"][:, 2] / np.float32(pitch)).astype(np.int64), geo.n_layers - 1)
    assert ((t["vol"] >> 1) == layer).all()
    ids = t["id_hi"].astype(np.uint64) << np.uint64(32) | t["id_lo"].astype(np.uint64)
    assert np.unique(ids).shape[0] == n                                             # distinct streams


def test_sweep_population_matches_config_4():
    span = 1 << 14
    for occ in (0.1, 0.9):
        pop = gen_sweep(occ, span=span)
        again = gen_sweep(occ, span=span)
        for k in range(3):
            p = pop[k]
            assert p["tracks"].tobytes() == again[k]["tracks"].tobytes()
            assert p["tracks"].shape[0] == round(occ * span)
            assert (np.diff(p["slots"].astype(np.int64)) > 0).all() and p["slots"].max() < span   # ascending, distinct
            f = p["forced"]
            assert 0.03 < f.mean() < 0.07                                            # 5 % spawn one secondary
            j = 0 if k < 2 else 2
            assert (p["tracks"]["nial"][f, j] == np.float32(1e-30)).all()
            assert (p["tracks"]["nial"][~f] == np.float32(1e6)).all()
    shuffled = gen_sweep(0.5, span=span, shuffled=True)[0]["slots"]
    assert (np.diff(shuffled.astype(np.int64)) < 0).any() and np.unique(shuffled).shape[0] == shuffled.shape[0]


def test_primaries_and_config_table():
    p = gen_primaries(16, 10.0)
    assert p.dtype.itemsize == 32 and (p["kind"] == 0).all() and (p["ekin"] == 10.0).all()
    assert (p["dir"] == np.float32([0, 0, 1])).all() and (p["pos"] == 0).all()
    assert CONFIGS["full"]["n_primaries"] == 1000 and CONFIGS["full"]["e_primary"] == 1000.0
    assert CONFIGS["heavy"]["n_primaries"] == 10000 and CONFIGS["heavy"]["capacity"] == 8 * 1024 * 1024
    assert CONFIGS["single_step"]["n_tracks"] == 1 << 24 and CONFIGS["sweep"]["span"] == 4 * 1024 * 1024
    assert geometry_for("tiny").n_layers == 4 and geometry_for("heavy").n_layers == 50
    assert tables_for("tiny").n_bins == 64 and tables_for("full").n_bins == 256
