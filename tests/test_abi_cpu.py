"""CPU-side checks of the boundary (no compute calls): the C-ABI library builds for sm_100a, loads, and
exports every symbol include/ls.h declares; the binding mirrors the header; the product package never
touches oracle/; the workload generator is deterministic and follows the BASELINE.json recipe."""
import ctypes
import os
import re

import numpy as np
import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _header_symbols():
    src = open(os.path.join(ROOT, "include", "ls.h")).read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    return sorted(set(re.findall(r"\b(ls_[a-z_0-9]+)\s*\(", src)))


def test_library_builds_and_exports_every_declared_symbol():
    from paper_2409_08090_b200 import binding
    from paper_2409_08090_b200.build import build
    path = build()
    assert os.path.exists(path)
    lib = ctypes.CDLL(path)
    declared = _header_symbols()
    assert "ls_plan" in declared and "ls_execute" in declared and "ls_destroy" in declared
    for name in declared:
        assert hasattr(lib, name), f"{name} declared in include/ls.h but not exported"
    assert sorted(binding.exported_symbols()) == declared, "binding and header disagree"
    # the pure-host entry point works without a device
    assert binding.ls_strerror(0) == "success"
    assert "invalid" in binding.ls_strerror(1)


def test_ls_opts_layout_matches_header():
    """Offsets and size of the ctypes mirror against what gcc computes from include/ls.h itself."""
    import subprocess, tempfile
    from paper_2409_08090_b200.binding import ls_opts
    names = [f[0] for f in ls_opts._fields_]
    prog = '#include <stdio.h>\n#include <stddef.h>\n#include "ls.h"\nint main(void){\n'
    for n in names:
        prog += f'  printf("{n} %zu\\n", offsetof(ls_opts, {n}));\n'
    prog += '  printf("sizeof %zu\\n", sizeof(ls_opts));\n  return 0;\n}\n'
    with tempfile.TemporaryDirectory() as d:
        src, exe = os.path.join(d, "o.c"), os.path.join(d, "o")
        with open(src, "w") as f:
            f.write(prog)
        subprocess.run(["gcc", "-I", os.path.join(ROOT, "include"), src, "-o", exe], check=True)
        out = dict(l.split() for l in subprocess.run([exe], check=True, capture_output=True, text=True).stdout.splitlines())
    for n in names:
        assert getattr(ls_opts, n).offset == int(out[n]), n
    assert ctypes.sizeof(ls_opts) == int(out["sizeof"])


def test_no_device_means_loud_failure_not_fallback():
    """Without a usable GPU ls_plan must return LS_ERR_CUDA (there is no CPU path)."""
    import torch
    if torch.cuda.is_available():
        pytest.skip("a device is present; the failure path is for the CPU box")
    from paper_2409_08090_b200 import binding
    with pytest.raises(binding.LsError) as ei:
        binding.ls_plan(100, 1000, 0.1, 0.1, 1e-9, binding.LS_F64, 1)
    assert ei.value.code == 3


def test_product_never_imports_the_oracle():
    pkg = os.path.join(ROOT, "paper_2409_08090_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".h", ".cuh", ".cpp", ".c")):
                txt = open(os.path.join(dirpath, f)).read()
                assert not re.search(r"^\s*(from|import)\s+oracle\b", txt, flags=re.M), f
                assert "ls_oracle" not in txt, f
    for f in os.listdir(os.path.join(ROOT, "oracle")):
        if f.endswith((".py", ".c")):
            txt = open(os.path.join(ROOT, "oracle", f)).read()
            assert not re.search(r"^\s*(from|import)\s+paper_2409_08090_b200\b", txt, flags=re.M), f


def test_workloads_follow_the_recipe():
    from paper_2409_08090_b200.workloads import compare_indices, make_workload, scaled_workload
    w1 = make_workload(1)
    assert w1.Nd == 1000 and w1.Nf == 12500 and w1.batch == 1 and w1.dtype == "f64" and w1.eps == 1e-9
    assert np.all(np.diff(w1.t) >= 0) and 0 <= w1.t.min() and w1.t.max() < 1000
    T = w1.t.max() - w1.t.min()
    assert w1.df == 1.0 / (5.0 * T) and w1.f0 == w1.df
    assert 0.5 <= w1.dy.min() and w1.dy.max() <= 1.5
    w1b = make_workload(1)
    assert np.array_equal(w1.t, w1b.t) and np.array_equal(w1.y, w1b.y) and np.array_equal(w1.dy, w1b.dy)
    w2 = make_workload(2)
    assert w2.Nd == 10_000 and w2.Nf == 125_000 and not np.all(np.diff(w2.t) >= 0)
    w4 = scaled_workload(4, 500, batch=7)
    assert w4.y.shape == (7, 500) and w4.dy.shape == (500,) and len(w4.injected) == 7
    w5 = scaled_workload(5, 20_000)
    assert w5.dtype == "f32" and w5.y.dtype == np.float32 and w5.dy.dtype == np.float32 and w5.t.dtype == np.float64
    night = np.floor(w5.t).astype(int)
    assert np.all((night % 365) < 219) and np.all(w5.t - night < 0.3)          # seasonal gap + 0.3-day windows
    ks = compare_indices(w2, 64)
    assert ks[0] == 0 and ks[-1] == w2.Nf - 1 and w2.Nf // 2 in ks and np.all(np.diff(ks) > 0)
    kc = int(round((1 / 23.1 - w2.f0) / w2.df))
    assert kc in ks
