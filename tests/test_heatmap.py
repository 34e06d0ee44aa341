"""Host-side rendering of the instrumented build's counters (heatmaps with a
selectable row size; per-field counts).  Pure CPU: synthetic counters in, files out."""
import numpy as np
import pytest

from paper_2302_08252_b200.heatmap import field_table_csv, rebin_rows, summarize, write_pgm


def test_rebin_rows_conserves_counts_and_checks_granularity():
    lines = np.arange(10, dtype=np.uint32)
    assert rebin_rows(lines, 128).tolist() == list(range(10))
    assert rebin_rows(lines, 256).tolist() == [1, 5, 9, 13, 17]
    assert rebin_rows(lines, 512).tolist() == [6, 22, 17] and rebin_rows(lines, 512).sum() == lines.sum()
    with pytest.raises(ValueError):
        rebin_rows(lines, 64)


def test_pgm_is_a_valid_p5_image_with_cold_rows_black(tmp_path):
    counts = np.zeros(1000, dtype=np.uint32)
    counts[10:20] = 5
    counts[500] = 1000
    w, h = write_pgm(counts, str(tmp_path / "a.pgm"), width=64)
    raw = (tmp_path / "a.pgm").read_bytes()
    header = b"P5\n64 16\n255\n"
    assert (w, h) == (64, 16) and raw.startswith(header) and len(raw) == len(header) + 64 * 16
    pix = np.frombuffer(raw[len(header):], dtype=np.uint8)
    assert pix[500] == 255 and (pix[10:20] > 0).all() and (pix[10:20] < 255).all()
    assert pix[:10].sum() == 0 and pix[1000:].sum() == 0          # untouched rows and padding are black
    write_pgm(np.zeros(5, dtype=np.uint32), str(tmp_path / "b.pgm"), width=4)   # all-cold buffer: no division by zero


def test_summary_and_field_table(tmp_path):
    lines = np.zeros((3, 64), dtype=np.uint32)
    slots = np.zeros((3, 256), dtype=np.uint32)
    lines[0, :8] = 3
    slots[0, :40] = 14
    slots[2, 200] = 1
    rw = np.arange(3 * 14 * 2, dtype=np.uint64).reshape(3, 14, 2)
    s = summarize(dict(lines=lines, slots=slots, field_rw=rw), row_bytes=256)
    assert s["electrons"] == {"rows": 32, "rows_touched": 4, "max_row_count": 6, "accesses": 24,
                              "slots_touched": 40, "highest_slot_touched": 40}
    assert s["photons"]["highest_slot_touched"] == 201 and s["positrons"]["slots_touched"] == 0
    names = ["f%d" % i for i in range(14)]
    field_table_csv(rw, names, str(tmp_path / "f.csv"))
    rows = (tmp_path / "f.csv").read_text().strip().split("\n")
    assert rows[0] == "kind,field,reads,writes" and len(rows) == 1 + 42
    assert rows[1] == "electrons,f0,0,1" and rows[-1] == "photons,f13,82,83"
