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
