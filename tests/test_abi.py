"""CPU-only checks of the boundary: the C-ABI library builds, loads and exports every symbol that
include/mlens.h declares; without a CUDA device every compute call fails loudly (no CPU fallback)."""
import ctypes
import os
import re

import numpy as np
import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def so():
    from paper_2506_02114_b200 import build
    return build.build()


def test_exports_every_declared_symbol(so):
    hdr = open(os.path.join(ROOT, "include", "mlens.h")).read()
    hdr = re.sub(r"/\*.*?\*/", "", hdr, flags=re.S)
    names = set(re.findall(r"\b(mlens_[a-z_0-9]+)\s*\(", hdr))
    assert {"mlens_field_create", "mlens_field_create_seeded", "mlens_shoot", "mlens_deflect",
            "mlens_grid_info", "mlens_field_get_stars", "mlens_field_destroy", "mlens_version"} <= names
    L = ctypes.CDLL(so)
    for n in names:
        assert hasattr(L, n), n
    L.mlens_version.restype = ctypes.c_int
    assert L.mlens_version() == 200
    # the roofline micro-benchmarks are a library of their own (include/mlens_bench.h), not part of the product ABI
    assert not hasattr(L, "mlens_bench_dfma") and not hasattr(L, "mlens_bench_atomics")
    bh = re.sub(r"/\*.*?\*/", "", open(os.path.join(ROOT, "include", "mlens_bench.h")).read(), flags=re.S)
    bnames = set(re.findall(r"\b(mlens_[a-z_0-9]+)\s*\(", bh))
    assert bnames == {"mlens_bench_dfma", "mlens_bench_atomics", "mlens_bench_shared_atomics",
                      "mlens_bench_atomics_pattern", "mlens_bench_shared_atomics_kind"}
    from paper_2506_02114_b200 import build
    B = ctypes.CDLL(build.BENCH_SO)
    for n in bnames:
        assert hasattr(B, n), n


def test_struct_sizes_match_header(so):
    # the ctypes mirrors must have the C layout: compile a tiny probe with gcc and compare sizeof
    import subprocess, tempfile
    from paper_2506_02114_b200 import mlens
    src = '#include <stdio.h>\n#include "mlens.h"\nint main(){printf("%zu %zu %zu %zu %zu %zu %zu\\n",' \
          'sizeof(mlens_field_desc),sizeof(mlens_seed_desc),sizeof(mlens_field_info),sizeof(mlens_shoot_desc),' \
          'sizeof(mlens_grid),sizeof(mlens_stats),sizeof(mlens_tree_view));return 0;}\n'
    with tempfile.TemporaryDirectory() as td:
        open(os.path.join(td, "p.c"), "w").write(src)
        subprocess.run(["gcc", "-I", os.path.join(ROOT, "include"), "-o", os.path.join(td, "p"), os.path.join(td, "p.c")], check=True)
        out = subprocess.run([os.path.join(td, "p")], check=True, capture_output=True, text=True).stdout.split()
    got = [ctypes.sizeof(c) for c in (mlens.FieldDesc, mlens.SeedDesc, mlens.FieldInfo, mlens.ShootDesc,
                                      mlens.Grid, mlens.Stats, mlens.TreeView)]
    assert got == [int(v) for v in out]


def test_no_cpu_fallback(so):
    import torch
    if torch.cuda.is_available():
        pytest.skip("a GPU is present")
    import paper_2506_02114_b200 as ml
    z = np.zeros(1)
    with pytest.raises(ml.MlensError, match="no CUDA device"):
        ml.Field.from_stars(0.4, 0.2, z, z, z, kappa_star=0.2, R=1.0)
    with pytest.raises(ml.MlensError):
        ml.bench_dfma()


def test_no_environment_knobs():
    """The library is configured through its C structs only ("plain C structs; no config files"): no getenv."""
    csrc = os.path.join(ROOT, "paper_2506_02114_b200", "csrc")
    for fn in os.listdir(csrc):
        assert "getenv" not in open(os.path.join(csrc, fn)).read(), fn


def test_product_does_not_import_oracle():
    pkg = os.path.join(ROOT, "paper_2506_02114_b200")
    for dirpath, _, files in os.walk(pkg):
        for fn in files:
            if fn.endswith((".py", ".cu", ".cuh", ".h")):
                txt = open(os.path.join(dirpath, fn)).read()
                assert "oracle" not in txt.replace("a-posteriori", ""), fn


def test_star_file_round_trip(tmp_path):
    """Star files: text and .npy round trips are bit-exact; comments, commas and bad rows."""
    import numpy as np
    from paper_2506_02114_b200.starfile import read_star_file, write_star_file
    rng = np.random.default_rng(3)
    x, y, m = rng.normal(size=50) * 100, rng.normal(size=50) * 100, rng.uniform(0.08, 1.0, 50)
    for name in ("stars.txt", "stars.npy"):
        p = tmp_path / name
        write_star_file(p, x, y, m)
        rx, ry, rm = read_star_file(p)
        assert np.array_equal(rx, x) and np.array_equal(ry, y) and np.array_equal(rm, m)
    p = tmp_path / "hand.txt"
    p.write_text("# x1 x2 m\n1.0, 2.0, 0.5  # first\n\n-3 4 1\n")
    rx, ry, rm = read_star_file(p)
    assert list(rx) == [1.0, -3.0] and list(ry) == [2.0, 4.0] and list(rm) == [0.5, 1.0]
    p.write_text("1 2 -1\n")
    with pytest.raises(ValueError):
        read_star_file(p)

