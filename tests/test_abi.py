"""-m "not gpu": the C-ABI library builds for sm_100a, loads, and exports every symbol that
include/landau.h declares.  No compute call is made (there is no GPU here)."""
import ctypes as C
import re
from pathlib import Path

import numpy as np
import pytest

ROOT = Path(__file__).resolve().parent.parent


@pytest.fixture(scope="module")
def binding():
    from paper_2212_00663_b200 import binding
    binding.load()
    return binding


def declared_symbols():
    text = (ROOT / "include" / "landau.h").read_text()
    text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)
    return sorted(set(re.findall(r"\b(landau_[a-z0-9_]+)\s*\(", text)))


def test_header_symbols_are_all_exported(binding):
    lib = binding.load()
    names = declared_symbols()
    assert len(names) >= 20
    for n in names:
        assert hasattr(lib, n), f"{n} declared in include/landau.h but not exported"
    assert sorted(binding.SYMBOLS) == names


def test_library_is_sm100a_only(binding):
    import subprocess
    out = subprocess.run(["cuobjdump", "-lelf", str(binding.library_path())], capture_output=True, text=True).stdout
    assert "sm_100a" in out
    assert not re.search(r"sm_(?!100a)\d+", out)


def test_create_fails_loudly_without_gpu(binding):
    import torch
    if torch.cuda.is_available():
        pytest.skip("a GPU is present")
    lib = binding.load()
    h = C.c_void_p()
    one = np.ones(1)
    rc = lib.landau_create(C.byref(h), 1, binding._hd(one), binding._hd(one), binding._hd(one), None)
    assert rc == binding.ECUDA and not h.value
    with pytest.raises(RuntimeError):
        binding.Landau([1.0], [1.0], [0.1])


def test_product_does_not_import_oracle():
    pkg = ROOT / "paper_2212_00663_b200"
    for p in list(pkg.rglob("*.py")) + list(pkg.rglob("*.cu*")) + list((ROOT / "include").glob("*.h")):
        t = p.read_text()
        assert "landau_ref" not in t and "import oracle" not in t and "from oracle" not in t, p
    for p in (ROOT / "oracle").glob("*"):
        if p.suffix in (".c", ".h", ".py"):
            t = p.read_text()
            assert "liblandau.so" not in t and "binding" not in t, p


def test_opts_struct_layout(binding):
    o = binding.Opts()
    binding.load().landau_default_opts(C.byref(o))
    assert (o.n_q, o.nu0, o.precision, o.pair_kernel, o.entropy_kernel, o.device) == (4, 1.0, 0, 0, 0, -1)


def test_cell_limits_in_the_header_are_the_ones_enforced(binding):
    """include/landau.h states the per-cell marker limits; landau_cells_max_markers is what landau_cells_run checks."""
    text = (ROOT / "include" / "landau.h").read_text()
    m = re.search(r"<= 1024 \(n_q <= 5\), (\d+) / (\d+) /\s*\*?\s*(\d+) at n_q = 6 / 7 / 8", text)
    assert m, "the limits sentence of landau_cells_run moved"
    assert [binding.cells_max_markers(q) for q in (2, 3, 4, 5)] == [1024] * 4
    assert [binding.cells_max_markers(q) for q in (6, 7, 8)] == [int(g) for g in m.groups()]
    assert binding.cells_max_markers(9) == 0 and binding.cells_max_markers(1) == 0
