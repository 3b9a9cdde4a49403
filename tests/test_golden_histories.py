"""The stored oracle histories (tests/golden/oracle_history_*.csv) are complete, self-describing and reproducible:
re-running the committed generator (which calls only oracle/) for the first steps of config 0 gives the stored rows."""
import re
import subprocess
import sys
from pathlib import Path

import numpy as np

GOLDEN = Path(__file__).resolve().parent / "golden"
ROOT = GOLDEN.parent.parent


def _read(path):
    lines = path.read_text().splitlines()
    body = [ln for ln in lines if not ln.startswith("#")]
    cols = body[0].split(",")
    rows = np.array([[float(x) for x in ln.split(",")] for ln in body[1:]])
    return lines, cols, rows


def test_golden_history_files_are_complete_and_name_their_command():
    files = sorted(GOLDEN.glob("oracle_history_c*_n*_s*.csv"))
    have = set()
    for f in files:
        cfg, nps, steps = map(int, re.match(r"oracle_history_c(\d+)_n(\d+)_s(\d+)", f.stem).groups())
        lines, cols, rows = _read(f)
        assert any("make_oracle_histories.py" in ln and f"--config {cfg}" in ln for ln in lines[:4]), f.name
        assert rows.shape == (steps + 1, len(cols)) and np.array_equal(rows[:, 0], np.arange(steps + 1)), f.name
        assert np.all(np.isfinite(rows[:, cols.index("K_0")])) and np.all(rows[1:, cols.index("iterations")] >= 1)
        # momentum (Eq. 26-27) is conserved by every iterate, converged or not
        P = rows[:, [i for i, c in enumerate(cols) if re.match(r"P[xyz]_\d", c)]]
        S = P.shape[1] // 3
        Ptot = P.reshape(len(rows), S, 3).sum(axis=1)
        assert np.abs(Ptot - Ptot[0]).max() <= 1e-12 * max(np.abs(P).max(), 1e-300), f.name
        have.add((cfg, nps))
    # full length c0, c1; first steps at full size and N_s = 2048 full length for c2, c3
    assert {(0, 256), (1, 4096), (2, 8192), (2, 2048), (3, 32768), (3, 2048)} <= have, have


def test_generator_reproduces_the_stored_config0_rows(tmp_path):
    out = subprocess.run([sys.executable, str(GOLDEN / "make_oracle_histories.py"), "--config", "0", "--steps", "2",
                          "--entropy-every", "1", "--threads", "2", "--out", str(tmp_path)],
                         capture_output=True, text=True, cwd=str(ROOT))
    assert out.returncode == 0, out.stderr
    _, cols_new, new = _read(tmp_path / "oracle_history_c0_n256_s2.csv")
    _, cols_old, old = _read(GOLDEN / "oracle_history_c0_n256_s10.csv")
    assert cols_new == cols_old
    skip = cols_old.index("oracle_seconds")
    keep = [i for i in range(len(cols_old)) if i != skip]
    np.testing.assert_allclose(new[:, keep], old[:3, keep], rtol=1e-13, atol=1e-15)
