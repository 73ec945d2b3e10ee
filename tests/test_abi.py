"""Host-side checks that need no GPU: the C-ABI library loads and exports every symbol that
include/ea.h declares; workspace sizing; the binding refuses to run without a device."""
import re
from pathlib import Path

import pytest

ROOT = Path(__file__).resolve().parents[1]


@pytest.fixture(scope="module")
def built():
    import __graft_entry__ as ge
    ge.build()
    import paper_1311_5582_b200 as pkg
    return pkg


def test_every_declared_symbol_is_exported(built):
    header = (ROOT / "include" / "ea.h").read_text()
    declared = set(re.findall(r"\b(ea_[a-z_]+)\s*\(", header))
    declared.discard("ea_handle")
    l = built.lib()
    assert declared, "no declarations found"
    for name in sorted(declared):
        assert hasattr(l, name), f"{name} declared in ea.h but not exported"
    assert declared == set(built.exported_symbols())


def test_workspace_bytes(built):
    l = built.lib()
    assert l.ea_workspace_bytes(5, 4, 1) == 0          # odd L
    assert l.ea_workspace_bytes(4, 100, 1) == 0        # too many temperatures
    n = l.ea_workspace_bytes(16, 24, 2048)
    spins = 24 * 64 * 4096 * 4
    coup = 3 * 64 * 4096 * 4
    assert spins + coup <= n <= spins + coup + (8 << 20)


def test_no_cpu_fallback(built):
    import torch
    if torch.cuda.is_available():
        pytest.skip("GPU present")
    import numpy as np
    with pytest.raises(built.EAError):
        built.EA(4, 2, 1, np.array([1.0, 0.5]), 1)
    # the raw C call fails as well (NULL handle), it does not compute on the CPU
    assert not built.lib().ea_create(4, 2, 1, np.array([1.0, 0.5]).ctypes.data, 1)
    assert b"no CUDA device" in built.lib().ea_last_error(None)


def test_product_does_not_touch_oracle():
    for path in (ROOT / "paper_1311_5582_b200").rglob("*"):
        if path.suffix in (".py", ".cu", ".cuh", ".h"):
            text = path.read_text()
            assert "import oracle" not in text and "from oracle" not in text and "ea_oracle" not in text
    for path in (ROOT / "oracle").rglob("*.py"):
        assert "paper_1311_5582_b200" not in path.read_text().replace("(paper_1311_5582_b200)", "")


def test_header_is_plain_c_and_the_c_example_links(built, tmp_path):
    """include/ea.h must compile as C (the boundary is a C ABI), and the C example must build and
    link against libea_b200.so with nothing but the header (it is run on the GPU box only)."""
    import subprocess
    inc = ROOT / "include"
    subprocess.check_call(["gcc", "-std=c99", "-Wall", "-Werror", "-pedantic", "-fsyntax-only", "-x", "c",
                           str(inc / "ea.h")])
    src = ROOT / "paper_1311_5582_b200" / "examples" / "ea_demo.c"
    exe = tmp_path / "ea_demo"
    subprocess.check_call(["gcc", "-std=c99", "-Wall", "-Werror", str(src), "-I", str(inc),
                           "-L", str(built.library_path().parent), "-lea_b200", "-lm",
                           f"-Wl,-rpath,{built.library_path().parent}", "-o", str(exe)])
    assert exe.exists()
