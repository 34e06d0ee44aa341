"""bench.py's reference arm (the oracle on host cores) runs without a GPU: check the JSON line it
prints against the keys the measurement contract names."""
import json
import os
import subprocess
import sys

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _run(extra_env=None, extra_args=()):
    env = {k: v for k, v in os.environ.items() if k not in ("RANK", "WORLD_SIZE", "LOCAL_RANK")}
    env.update(extra_env or {})
    out = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--steps", "2",
                          "--warmup", "1", "--tracks", "65536", *extra_args], capture_output=True, text=True, env=env,
                         timeout=600)
    assert out.returncode == 0, out.stderr[-2000:]
    return out.stdout.strip()


def test_reference_arm_prints_one_contract_line():
    text = _run()
    lines = [l for l in text.split("\n") if l.strip()]
    assert len(lines) == 1
    d = json.loads(lines[0])
    assert d["impl"] == "reference" and d["metric"] == "track-steps/sec" and d["unit"] == "track-steps/s"
    assert d["higher_is_better"] is True and d["steps"] == 2 and d["warmup"] == 1 and d["vs_baseline"] is None
    assert d["value"] > 1e5 and d["ms_per_step"] > 0 and d["dtype"] == "f32" and d["data"] == "synthetic"
    assert "workload" in d["config"] and "model" not in d["config"]
    cb = d["cpu_baseline"]
    assert cb["kind"] == "oracle" and cb["cores"] == 1 and cb["value"] == d["value"] and "sample" in cb
    assert cb["host_cores"] == os.cpu_count() and d["n_gpus"] == 1
    assert d["e2e"] == {"value": d["value"], "unit": d["unit"], "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0}


def test_reference_arm_other_ranks_stay_silent():
    assert _run({"RANK": "1", "WORLD_SIZE": "2", "LOCAL_RANK": "1"}) == ""


def test_gpus_flag_launches_the_ranks_itself():
    """`python bench.py --gpus 2` outside torchrun runs two ranks (127.0.0.1 rendezvous); rank 0 alone
    prints, and n_gpus is the number of ranks that ran."""
    lines = [l for l in _run(extra_args=("--gpus", "2")).split("\n") if l.strip().startswith("{")]
    assert len(lines) == 1
    d = json.loads(lines[0])
    assert d["impl"] == "reference" and d["n_gpus"] == 2


import pytest


@pytest.mark.gpu
def test_gpu_arm_prints_one_contract_line():
    """The product arm at a reduced population: every key of the measurement contract is there."""
    out = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--steps", "3", "--warmup", "3",
                          "--tracks", "262144", "--layout", "aosoa32"], capture_output=True, text=True, timeout=600)
    assert out.returncode == 0, out.stderr[-2000:]
    lines = [l for l in out.stdout.split("\n") if l.strip()]
    assert len(lines) == 1
    d = json.loads(lines[0])
    for k in ("metric", "value", "unit", "n_gpus", "steps", "warmup", "ms_per_step", "higher_is_better", "scaling",
              "vs_baseline", "dtype", "data", "config", "clocks", "gpu_launches", "e2e", "roofline", "cpu_baseline"):
        assert k in d, k
    assert d["n_gpus"] == 1 and d["steps"] == 3 and d["gpu_launches"] == 3 and d["scaling"] == "weak"
    assert d["config"]["layout"] == "aosoa32" and "workload" in d["config"]
    rf = d["roofline"]
    assert rf["bound"] == "hbm" and rf["unit"] == "GB/s" and abs(rf["frac"] - rf["achieved"] / rf["peak"]) < 1e-12
    assert rf["traffic"] is None                       # the ncu figure belongs to the full-size workload only
    e = d["e2e"]
    assert e["h2d_bytes_per_step"] == 56 * 262144 and e["d2h_bytes_per_step"] > 56 * 262144 and e["value"] < d["value"]
    cb = d["cpu_baseline"]
    assert cb["kind"] == "oracle" and cb["cores"] == 1 and cb["value"] > 1e5 and cb["host_cores"] >= 1
    assert "showers" not in d and "sweep" not in d      # reduced population: headline only
    p = d["parity_full_size"]
    assert p["counts_bit_exact"] and p["tracks_with_another_fate"] == 0 and p["tracks_with_any_word_differing"] == 0
    assert set(d["clocks"]) >= {"sm_mhz", "sm_max_mhz", "reasons"}


@pytest.mark.gpu
def test_gpu_arm_two_ranks_plumbing_on_one_device():
    """`bench.py --gpus 2` launches its two ranks, shards the single-step population by rank (weak
    scaling, max over ranks) and the showers by primaries (one all-reduce of the tallies).  On this
    one-GPU box both ranks run on cuda:0 over gloo (ADEPT_BENCH_ONE_DEVICE: plumbing test, not a timing)."""
    env = {k: v for k, v in os.environ.items() if k not in ("RANK", "WORLD_SIZE", "LOCAL_RANK")}
    env["ADEPT_BENCH_ONE_DEVICE"] = "1"
    out = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--gpus", "2", "--steps", "3", "--warmup", "3",
                          "--tracks", "262144", "--layout", "aosoa32", "--extras", "showers"],
                         capture_output=True, text=True, timeout=900, env=env)
    assert out.returncode == 0, out.stderr[-3000:]
    lines = [l for l in out.stdout.split("\n") if l.strip().startswith("{")]
    assert len(lines) == 1
    d = json.loads(lines[0])
    assert d["n_gpus"] == 2 and d["scaling"] == "weak" and "cpu_baseline" not in d
    assert d["config"]["parallelism"].startswith("independent track shards")
    sh = d["showers"]["full_sharded"]
    assert sh["scaling"] == "strong" and sh["iterations"] == 172 and sh["track_steps"] == 6999724   # config 2, summed over the ranks


def _synthetic_full_result():
    """A result dict of the shape run_gpu builds at the full population: five shower blocks with their
    50-bin deposits, a 40-cell sweep with per-field counts -- tens of kilobytes before compaction."""
    import bench
    fields = ("pos.x", "pos.y", "pos.z", "dir.x", "dir.y", "dir.z", "ekin", "nial.0", "nial.1", "nial.2", "vol", "id_lo", "id_hi", "step")
    shower = lambda: {"value": 4.123456789e9, "unit": "track-steps/s", "ms_per_run": 1.7123456, "ms_min": 1.69876543, "runs": 3,
                      "iterations": 172, "track_steps": 6999724, "us_per_iteration": 9.912345, "showers_per_s": 5.8e5,
                      "layout": "aosoa32", "scheme": "dense", "secondaries": [1, 2, 3], "edep_layer_MeV": [1234.56789012345] * 50,
                      "cpu_baseline": {"value": 6.1e6, "cores": 1, "kind": "oracle", "sample": "x" * 60, "seconds": 1.1},
                      "parity_full_size": {"counts_bit_exact": True, "edep_layer_rel_err": 1.2345e-9, "e_escaped_rel_err": 0.0},
                      "same_counts_as_dense": True}
    cells = []
    for occ in (0.1, 0.3, 0.5, 0.7, 0.9):
        for scheme in ("dense", "sparse"):
            for layout in ("aos", "soa", "aosoa32", "hc16"):
                c = {"occupancy": occ, "scheme": scheme, "layout": layout, "tracks": 5662310, "ms_per_step": 0.333123456,
                     "ms_min": 0.33, "track_steps_per_s": 1.7e10, "secondaries": [1, 2, 3], "slots_used": [4, 5, 6],
                     "algorithmic_bytes": 1234567890,
                     "roofline": {"bound": "hbm", "achieved": 4567.891234, "peak": 6551.7, "unit": "GB/s", "frac": 0.6972345,
                                  "traffic": None, "traffic_source": None},
                     "section_share": {n: 0.1666 for n in bench.SECTION_NAMES}, "alloc_compaction_ms": 0.0712345,
                     "alloc_ms": 0.05, "store_ms": 0.02}
                if occ == 0.5:
                    c.update(field_reads={f: 5662310 for f in fields}, field_writes={f: 4123456 for f in fields},
                             lines_touched=1234567, slots_touched=5662310, bytes_touched_per_track_step=125.123456,
                             line_bytes=158024576, line_bytes_over_algorithmic=1.2345678)
                cells.append(c)
    lay = lambda: {"ms_per_step": 0.41612345, "ms_min": 0.414, "ms_median": 0.416, "track_steps_per_s": 4.03e10,
                   "algorithmic_bytes_per_launch": 2032800000, "algorithmic_GBps": 4885.123, "survivors_plus_secondaries": 19523553}
    return {
        "metric": "track-steps/sec", "value": 4.0312345e10, "unit": "track-steps/s", "n_gpus": 1, "steps": 20, "warmup": 5,
        "ms_per_step": 0.41612345, "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f32",
        "data": "synthetic", "config": {"workload": "w" * 160, "layout": "aosoa32", "scheme": "dense", "l2": "l" * 120},
        "clocks": {"sm_mhz": 1965.0, "sm_max_mhz": 1965.0, "reasons": [], "samples": 100}, "gpu_launches": 20,
        "e2e": {"value": 4.2e8, "unit": "track-steps/s", "h2d_bytes_per_step": 939524096, "d2h_bytes_per_step": 1093319480,
                "steps": 10, "ms_min": 39.1, "ms_median": 39.5, "counts_only": {"value": 9e8, "unit": "track-steps/s", "what": "c" * 70},
                "what": "e" * 80},
        "roofline": {"bound": "hbm", "achieved": 4885.1, "peak": 6551.7, "unit": "GB/s", "frac": 0.7456, "traffic": 1.989e9,
                     "traffic_source": "t" * 60, "peak_source": "p" * 40, "kernel": "k" * 60, "bytes_per_launch": 2032800000},
        "cpu_baseline": {"value": 6.0e6, "unit": "track-steps/s", "cores": 1, "host_cores": 64, "kind": "oracle", "sample": "s" * 70,
                         "seconds": 2.8},
        "parity_full_size": {"counts_bit_exact": True, "tracks_compared": 19523553, "tracks_with_another_fate": 0,
                             "tracks_with_any_word_differing": 0, "branch_disagreement_rate": 0.0, "edep_rel_err": 1e-9},
        "layouts": {l: lay() for l in ("aosoa32", "aosoa64", "soa16", "hc16", "soa", "aos")},
        "showers": {n: shower() for n in ("full", "heavy", "full_physics2", "full_sparse_recycle", "heavy_sparse_recycle")},
        "sweep": {"workload": "x", "peak_source": "y", "sections": "z" * 300,
                  "best": {"occupancy": 0.9, "scheme": "dense", "layout": "aosoa32", "ms_per_step": 0.2, "track_steps_per_s": 2.8e10},
                  "cells": cells},
        "extras_file": "bench_extras.json",
    }


def test_contract_line_of_a_full_size_result_is_compact_and_complete():
    """What the driver parses is ONE line, the last of stdout, short enough to survive its bounded tail
    (round 2 lost its measurement to a line of tens of kilobytes): the contract keys are all there,
    the extras only as summaries, BASELINE.json configs[3]'s per-field counts among them."""
    import bench
    full = _synthetic_full_result()
    assert len(json.dumps(full)) > 4 * bench.LINE_LIMIT        # the thing that must not be printed
    text = json.dumps(bench.contract_line(full))
    assert len(text) < bench.LINE_LIMIT, len(text)
    d = json.loads(text)
    for k in ("metric", "value", "unit", "n_gpus", "steps", "warmup", "ms_per_step", "higher_is_better", "scaling",
              "vs_baseline", "dtype", "data", "config", "clocks", "gpu_launches", "e2e", "roofline", "cpu_baseline",
              "parity_full_size"):
        assert d[k] == full[k], k
    assert d["showers"]["full"]["counts_bit_exact"] is True and d["showers"]["full"]["iterations"] == 172
    assert "edep_layer_MeV" not in d["showers"]["full"] and "cells" not in d["sweep"]
    sw = d["sweep"]
    assert sw["occupancies"] == [0.1, 0.3, 0.5, 0.7, 0.9] and sw["layouts"] == ["aos", "soa", "aosoa32", "hc16"]
    for scheme in ("dense", "sparse"):
        assert len(sw[scheme]["ms_per_step"]) == 4 and all(len(r) == 5 for r in sw[scheme]["roofline_frac"])
        fc = sw[scheme]["field_counts"]
        assert fc["layout"] == "aosoa32" and len(fc["reads"]) == len(fc["writes"]) == len(sw["field_names"]) == 14
        assert set(sw[scheme]["line_bytes_over_algorithmic"]) == {"aos", "soa", "aosoa32", "hc16"}
    assert d["layouts_ms_per_step"]["aos"] == 0.41612 and d["extras_file"] == "bench_extras.json"


def test_emit_prints_the_contract_line_last_and_writes_the_extras(tmp_path, monkeypatch, capsys):
    import bench
    monkeypatch.setattr(bench, "EXTRAS_FILE", str(tmp_path / "bench_extras.json"))
    full = _synthetic_full_result()
    bench.emit(full)
    cap = capsys.readouterr()
    lines = [l for l in cap.out.split("\n") if l.strip()]
    assert len(lines) == 1 and len(lines[0]) < bench.LINE_LIMIT and json.loads(lines[0])["value"] == full["value"]
    assert not any(l.lstrip().startswith("{") for l in cap.err.split("\n"))
    kept = json.load(open(tmp_path / "bench_extras.json"))
    assert len(kept["sweep"]["cells"]) == 40 and len(kept["showers"]["heavy"]["edep_layer_MeV"]) == 50


@pytest.mark.gpu
@pytest.mark.slow
def test_the_drivers_exact_command_ends_with_the_contract_line():
    """`python bench.py --gpus 1 --steps 20 --warmup 5`, as the driver runs it: of everything the run
    writes (stdout and stderr together), the last JSON-parsable line is the contract line, it is the last
    line of stdout, and nothing on stderr looks like JSON."""
    out = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--gpus", "1", "--steps", "20", "--warmup", "5"],
                         capture_output=True, text=True, timeout=1500)
    assert out.returncode == 0, out.stderr[-3000:]
    assert not any(l.lstrip().startswith("{") for l in out.stderr.split("\n"))
    stdout_lines = [l for l in out.stdout.split("\n") if l.strip()]
    parsable = []
    for l in (out.stdout + "\n" + out.stderr).split("\n"):
        try:
            parsable.append(json.loads(l))
        except ValueError:
            pass
    d = parsable[-1]
    assert isinstance(d, dict) and d == json.loads(stdout_lines[-1]) and len(stdout_lines[-1]) < 8192
    assert d["metric"] == "track-steps/sec" and d["value"] > 1e10 and d["steps"] == 20 and d["warmup"] == 5
    assert d["roofline"]["frac"] > 0.5 and d["cpu_baseline"]["kind"] == "oracle" and d["e2e"]["value"] > 0
    assert d["e2e"]["steps"] >= 10 and d["parity_full_size"]["counts_bit_exact"]
    assert d["showers"]["full"]["counts_bit_exact"] and d["showers"]["full"]["iterations"] == 172
    for scheme in ("dense", "sparse"):
        fc = d["sweep"][scheme]["field_counts"]
        assert sum(fc["reads"]) > 0 and sum(fc["writes"]) > 0
    for ph in ("physics1", "physics2"):   # the same step under the extended rule sets, timed and compared at full size
        b = d["single_step_physics"][ph]
        assert b["counts_bit_exact"] and b["tracks_with_any_word_differing"] == 0 and 0.2 < b["roofline_frac"] < 1.0
    extras = json.load(open(os.path.join(ROOT, d["extras_file"])))
    assert len(extras["sweep"]["cells"]) == 40
