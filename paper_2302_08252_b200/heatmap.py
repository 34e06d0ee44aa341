"""Access traces and heatmaps of an instrumented run (the paper's Trace / Heatmap mappings).

PAPER.md:115, 123: per-field read and write counts (Fig. 5); accesses per memory
row with a selectable row size, run with "-particles 25 -batch 5" because the counters are large
(Fig. 6-8); track slots touched (2044 dense against 45509 sparse).  The counting is
done on the device by the instrumented instantiation of the step kernel (`instrument=True`,
`adept_read_counters`); this module only turns the counters into files: CSV tables and binary PGM
images (one grey value per row, no graphics stack involved).

  python -m paper_2302_08252_b200.heatmap --out DIR [--primaries 25] [--batch 5] [--energy 10000]
         [--layout aos] [--scheme sparse|dense] [--capacity 262144] [--row-bytes 128]
"""
from __future__ import annotations

import argparse
import json
import os

import numpy as np

KIND_NAMES = ("electrons", "positrons", "photons")


def rebin_rows(lines: np.ndarray, row_bytes: int) -> np.ndarray:
    """Counts per 128-byte line -> counts per row of `row_bytes` (a multiple of 128: cache line,
    several lines, a track tile ...; "the row size can be chosen")."""
    if row_bytes % 128 or row_bytes <= 0:
        raise ValueError("row size must be a positive multiple of the 128-byte counting granularity")
    k = row_bytes // 128
    n = (lines.shape[0] + k - 1) // k
    padded = np.zeros(n * k, dtype=np.uint64)
    padded[:lines.shape[0]] = lines
    return padded.reshape(n, k).sum(axis=1)


def write_pgm(counts: np.ndarray, path: str, width: int = 512, log_scale: bool = True) -> tuple[int, int]:
    """One pixel per row, `width` pixels per image line, 0 = never touched, 255 = hottest row.
    Binary PGM (P5).  Returns (width, height)."""
    c = np.asarray(counts, dtype=np.float64)
    if log_scale:
        c = np.log1p(c)
    top = c.max() if c.size and c.max() > 0 else 1.0
    pix = np.zeros(((c.size + width - 1) // width) * width, dtype=np.uint8)
    pix[:c.size] = np.where(c > 0, np.maximum(1, np.round(255.0 * c / top)), 0).astype(np.uint8)
    h = pix.size // width
    with open(path, "wb") as f:
        f.write(b"P5\n%d %d\n255\n" % (width, h))
        f.write(pix.tobytes())
    return width, h


def field_table_csv(field_rw: np.ndarray, field_names, path: str) -> None:
    """[3][14][2] counters -> CSV: kind, field, reads, writes (Fig. 5's bars as numbers)."""
    with open(path, "w") as f:
        f.write("kind,field,reads,writes\n")
        for k, kn in enumerate(KIND_NAMES):
            for i, fn in enumerate(field_names):
                f.write("%s,%s,%d,%d\n" % (kn, fn, int(field_rw[k, i, 0]), int(field_rw[k, i, 1])))


def summarize(counters: dict, row_bytes: int = 128) -> dict:
    """The numbers the paper reads off its heatmaps: rows touched, hottest row, slots used."""
    out = {}
    for k, kn in enumerate(KIND_NAMES):
        rows = rebin_rows(counters["lines"][k], row_bytes)
        slots = counters["slots"][k]
        out[kn] = {"rows": int(rows.shape[0]), "rows_touched": int((rows > 0).sum()),
                   "max_row_count": int(rows.max()) if rows.size else 0,
                   "accesses": int(rows.sum()), "slots_touched": int((slots > 0).sum()),
                   "highest_slot_touched": int(np.nonzero(slots)[0].max()) + 1 if (slots > 0).any() else 0}
    return out


def main() -> None:
    ap = argparse.ArgumentParser(description=__doc__.split("\n")[0])
    ap.add_argument("--out", required=True)
    ap.add_argument("--primaries", type=int, default=25)
    ap.add_argument("--batch", type=int, default=5)
    ap.add_argument("--energy", type=float, default=1.0e4, help="MeV")
    ap.add_argument("--layout", default="aos")
    ap.add_argument("--scheme", default="sparse", choices=["sparse", "dense"])
    ap.add_argument("--capacity", type=int, default=1 << 18)
    ap.add_argument("--row-bytes", type=int, default=128)
    ap.add_argument("--seed", type=int, default=5)
    a = ap.parse_args()
    from workloads import gen_primaries, geometry_for, tables_for
    from . import FIELD_NAMES, Context
    os.makedirs(a.out, exist_ok=True)
    ctx = Context(geometry_for("heavy"), tables_for("heavy"), layout=a.layout, scheme=a.scheme,
                  capacity=a.capacity, seed=a.seed, batch_primaries=a.batch, instrument=True)
    ctx.inject(gen_primaries(a.primaries, a.energy))
    res = ctx.run()
    cnt = ctx.read_counters()
    ctx.destroy()
    tag = "%s_%s" % (a.scheme, a.layout)
    field_table_csv(cnt["field_rw"], FIELD_NAMES, os.path.join(a.out, "fields_%s.csv" % tag))
    for k, kn in enumerate(KIND_NAMES):
        write_pgm(rebin_rows(cnt["lines"][k], a.row_bytes), os.path.join(a.out, "rows_%s_%s.pgm" % (tag, kn)))
        write_pgm(cnt["slots"][k], os.path.join(a.out, "slots_%s_%s.pgm" % (tag, kn)))
    s = summarize(cnt, a.row_bytes)
    s["run"] = {"primaries": a.primaries, "batch": a.batch, "energy_MeV": a.energy, "layout": a.layout,
                "scheme": a.scheme, "capacity": a.capacity, "row_bytes": a.row_bytes,
                "iterations": res["iterations"], "track_steps": [int(x) for x in res["steps"]],
                "slots_used": [int(x) for x in res["slots_used"]]}
    with open(os.path.join(a.out, "summary_%s.json" % tag), "w") as f:
        json.dump(s, f, indent=1)
    print(json.dumps(s))


if __name__ == "__main__":
    main()
