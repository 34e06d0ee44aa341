"""bench.py's host-side helpers (no GPU): the committed ncu traffic table is what `roofline.traffic`
comes from, and the algorithmic byte counts of the sweep cells are the ones DESIGN.md §7.3 states."""
import importlib.util
import os

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _bench():
    spec = importlib.util.spec_from_file_location("bench_module", os.path.join(ROOT, "bench.py"))
    m = importlib.util.module_from_spec(spec)
    spec.loader.exec_module(m)
    return m


def test_traffic_comes_from_the_committed_table():
    b = _bench()
    nbytes, src = b.ncu_traffic("single_step", "aosoa32", "dense")
    rows = [l.strip().split(",") for l in open(os.path.join(ROOT, "profiles", "ncu_traffic.csv"))
            if l.strip() and not l.startswith("#")]
    last = [r for r in rows[1:] if r[0] == "single_step" and r[1] == "aosoa32" and r[2] == "dense"][-1]
    assert nbytes == float(last[6]) + float(last[7]) and last[4] in src and last[5] in src
    assert 1.9e9 < nbytes < 2.1e9                                    # ~ the algorithmic 2.03 GB: nothing is re-read
    assert b.ncu_traffic("single_step", "aos", "sparse") == (None, None)
    assert b.ncu_traffic("sweep_0.9", "aos", "sparse")[0] > 1.5e9


def test_sweep_bytes_are_the_stated_algorithmic_bytes():
    b = _bench()
    n, surv, sec = 1000, 900, 50
    assert b.sweep_bytes("dense", "soa", n, surv, sec) == 56 * (n + surv + sec)
    assert b.sweep_bytes("dense", "aos", n, surv, sec) == 64 * (n + surv + sec)
    assert b.sweep_bytes("sparse", "aos", n, surv, sec) == n * 68 + surv * 68 + sec * 68
    assert b.sweep_bytes("sparse", "hc16", n, surv, sec) == n * 60 + surv * 36 + sec * 60
    assert b.sweep_bytes("sparse", "soa16", n, surv, sec) == n * 60 + surv * 60 + sec * 60
    assert b.sweep_bytes("sparse", "aosoa32", n, surv, sec) == n * 60 + surv * 36 + sec * 60
    peak, src = b.measured_peak()
    assert 5000 < peak < 9000 and ("measured" in src or "fallback" in src)
