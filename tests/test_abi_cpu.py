"""CPU-side checks of the boundary: the C-ABI library builds, loads and exports every symbol the
header declares; the binding refuses to run without a GPU (no CPU fallback); the product package
does not import the oracle."""
import ast
import re
from pathlib import Path

import pytest

ROOT = Path(__file__).resolve().parent.parent


def test_library_builds_and_exports_every_declared_symbol():
    from paper_1709_06999_b200 import build
    build.build()
    import paper_1709_06999_b200 as g
    lib = g.load_library()
    header = (ROOT / "include" / "galario_b200.h").read_text()
    names = sorted(set(re.findall(r"\b(gal_[a-z0-9_]+)\s*\(", header)))
    assert len(names) >= 25
    for n in names:
        assert hasattr(lib, n), f"{n} declared in the header but not exported"
    assert lib.gal_strerror(0) == b"ok"
    assert lib.gal_strerror(-1) == b"invalid argument"


def test_no_cpu_fallback_without_gpu():
    import torch
    import paper_1709_06999_b200 as g
    if torch.cuda.is_available():
        pytest.skip("GPU present")
    with pytest.raises(g.GalarioError):
        g.Plan(256)
    with pytest.raises(g.GalarioError):
        g.sampleImage(torch.zeros(8, 8, dtype=torch.float64), 1e-7, torch.zeros(3, dtype=torch.float64),
                      torch.zeros(3, dtype=torch.float64))


def _imports(path):
    mods = []
    for node in ast.walk(ast.parse(path.read_text())):
        if isinstance(node, ast.Import):
            mods += [a.name for a in node.names]
        elif isinstance(node, ast.ImportFrom):
            mods.append(node.module or "")
    return [m.split(".")[0] for m in mods]


def test_product_never_imports_oracle_and_oracle_never_imports_product():
    for f in (ROOT / "paper_1709_06999_b200").rglob("*.py"):
        assert "oracle" not in _imports(f), f"{f} imports the oracle"
    for f in (ROOT / "oracle").rglob("*.py"):
        assert "paper_1709_06999_b200" not in _imports(f), f"{f} imports the product"
    inc = re.compile(r'#\s*include\s*[<"]([^>"]+)[>"]')
    for f in (ROOT / "paper_1709_06999_b200" / "csrc").iterdir():
        assert not any("oracle" in h for h in inc.findall(f.read_text())), f
    for h in inc.findall((ROOT / "oracle" / "galario_oracle.cpp").read_text()):
        assert "/" not in h and not h.endswith((".cuh", "galario_b200.h")), h     # standard headers only


def test_workloads_shapes_and_determinism():
    import numpy as np
    from paper_1709_06999_b200 import workloads as W
    a, b = W.config(0), W.config(0)
    assert a.nxy == 256 and a.M == 10_000 and a.image.shape == (256, 256)
    assert np.array_equal(a.u, b.u) and np.array_equal(a.image, b.image) and np.array_equal(a.re_obs, b.re_obs)
    assert abs(a.image.sum() - 1.17) < 1e-9              # 1 Jy Gaussian + 0.10 + 0.05 + 0.02 point sources
    assert np.abs(a.u).max() < 0.45 / a.dxy and np.allclose(a.w, 1e6)
    c1 = W.config(1, nxy=128, M=1000, nr=300)
    assert c1.entry == "chi2Profile" and c1.profile.shape == (300,) and c1.dRA == 0.0 and c1.dDec == 0.0
    c4 = W.config(4, nxy=64, M=500, C=3)
    assert c4.image.shape == (3, 64, 64) and c4.u.shape == (3, 500) and c4.entry == "chi2ImageBatch"
    f = a.as_f32()
    assert f.image.dtype == np.float32 and f.u.dtype == np.float32 and f.precision == "f32"
