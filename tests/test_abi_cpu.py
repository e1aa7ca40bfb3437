"""CPU-side checks of the boundary: libpakr.so builds for sm_100a, loads without a GPU and exports
every function include/pakr.h declares; the ctypes structs match the header's field order; the
workload generator is deterministic and keeps start/goal clear of obstacles (P30)."""
import ctypes
import os
import re

import numpy as np
import pytest

from paper_2607_03987_b200 import workloads as wl

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _declared_functions():
    text = open(os.path.join(ROOT, "include", "pakr.h")).read()
    text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)
    return sorted(set(re.findall(r"\b(pakr_[a-z0-9_]+)\s*\(", text)))


def test_library_exports_every_declared_symbol():
    from paper_2607_03987_b200 import pakr
    names = _declared_functions()
    assert set(names) == set(pakr.EXPORTS), names
    L = ctypes.CDLL(pakr.build())
    for n in names:
        assert hasattr(L, n), n


def test_measurement_support_is_a_library_of_its_own():
    """The roofline microbenchmark is not part of the product ABI: libpakr.so does not export it, libpakr_peak.so does."""
    from paper_2607_03987_b200 import pakr, peak
    assert not hasattr(ctypes.CDLL(pakr.build()), "pakr_measure_fp32_peak")
    assert hasattr(ctypes.CDLL(peak.build()), "pakr_measure_fp32_peak")
    assert "pakr_measure_fp32_peak" not in open(os.path.join(ROOT, "include", "pakr.h")).read()


def test_sass_is_sm100a_with_tma():
    """The built library carries sm_100a SASS and the NN scan's bulk copies are TMA (UBLKCP)."""
    from paper_2607_03987_b200 import pakr
    import subprocess
    so = pakr.build()
    out = subprocess.run(["/usr/local/cuda/bin/cuobjdump", "-sass", so], capture_output=True, text=True).stdout
    assert "sm_100a" in out
    assert "UBLKCP" in out


_STRUCTS = {"pakr_problem": "_Problem", "pakr_tree_layout": "_TreeLayout", "pakr_plan_opts": "_PlanOpts",
            "pakr_stats": "_Stats", "pakr_result": "_Result", "pakr_step_args": "_StepArgs"}


def _header_fields(name):
    text = open(os.path.join(ROOT, "include", "pakr.h")).read()
    body = re.search(r"typedef struct \{((?:(?!typedef struct).)*?)\} %s;" % name, text, flags=re.S).group(1)
    body = re.sub(r"/\*.*?\*/", "", body, flags=re.S)
    fields = []
    for decl in body.split(";"):
        decl = decl.strip()
        if not decl:
            continue
        names = re.sub(r"^(const\s+)?\w+\s*\*?", "", decl, count=1)
        fields += [re.sub(r"\[.*", "", n).strip(" *") for n in names.split(",")]
    return fields


@pytest.mark.parametrize("cname", sorted(_STRUCTS))
def test_struct_field_order_matches_header(cname):
    from paper_2607_03987_b200 import pakr
    assert _header_fields(cname) == [f[0] for f in getattr(pakr, _STRUCTS[cname])._fields_]


def test_struct_layout_matches_a_c_compiler(tmp_path):
    """include/pakr.h is plain C; sizeof / offsetof of every struct as gcc lays it out equal the ctypes mirrors."""
    import subprocess
    from paper_2607_03987_b200 import pakr
    lines = ['#include <stdio.h>', '#include <stddef.h>', '#include "pakr.h"', 'int main(void) {']
    for cname in sorted(_STRUCTS):
        lines.append('printf("%s %%zu\\n", sizeof(%s));' % (cname, cname))
        for f in _header_fields(cname):
            lines.append('printf("%s.%s %%zu\\n", offsetof(%s, %s));' % (cname, f, cname, f))
    lines += ['return 0; }']
    src = tmp_path / "abi.c"
    src.write_text("\n".join(lines))
    exe = tmp_path / "abi"
    subprocess.check_call(["gcc", "-std=c99", "-Wall", "-Werror", "-I", os.path.join(ROOT, "include"), "-o", str(exe), str(src)])
    got = dict(l.split() for l in subprocess.run([str(exe)], capture_output=True, text=True, check=True).stdout.splitlines())
    for cname, pyname in _STRUCTS.items():
        st = getattr(pakr, pyname)
        assert int(got[cname]) == ctypes.sizeof(st), cname
        for f, _ in st._fields_:
            assert int(got[f"{cname}.{f}"]) == getattr(st, f).offset, (cname, f)


def test_create_without_gpu_fails_loudly():
    import torch
    if torch.cuda.is_available():
        pytest.skip("GPU present")
    from paper_2607_03987_b200 import pakr
    p, _ = wl.config1()
    with pytest.raises(pakr.PakrError):
        pakr.Planner(p)


@pytest.mark.parametrize("name", ["C1", "C2", "C3", "C4", "C5", "N1", "N2", "N3"])
def test_workloads_deterministic_and_clear(name):
    a, cfg = wl.CONFIGS[name]()
    b, _ = wl.CONFIGS[name]()
    np.testing.assert_array_equal(a.obstacles, b.obstacles)
    assert a.obstacles.dtype == np.float32 and a.start.dtype == np.float32
    ps, g = a.start[:a.pos_dim].astype(np.float64), a.goal_center.astype(np.float64)
    if a.obstacle_type == wl.OBS_AABB:
        lo, hi = a.obstacles[:, :a.pos_dim], a.obstacles[:, a.pos_dim:]
        for q, clear in ((ps, 0.5), (g, 0.5 + a.goal_radius)):
            d = np.linalg.norm(np.maximum(np.maximum(lo - q, q - hi), 0), axis=1)
            assert d.min() > clear - 1e-6
        assert np.all(hi - lo >= 0.5 - 1e-6) and np.all(hi - lo <= 2.0 + 1e-6)
    else:
        for q, clear in ((ps[:2], 0.5), (g[:2], 0.5 + a.goal_radius)):
            d = np.linalg.norm(a.obstacles[:, :2] - q, axis=1) - a.obstacles[:, 2]
            assert d.min() > clear - 1e-6
    expected = {"C1": 8, "C2": 32, "C3": 64, "C4": 128, "C5": 128, "N1": 32, "N2": 40, "N3": 128}[name]
    assert a.n_obstacles == expected
    assert cfg.B >= 1 and cfg.K >= 1


def test_random_tree_invariants():
    p, _ = wl.config3()
    t = wl.random_tree(p, 500, seed=1)
    assert t["parents"][0] == -1 and np.all(t["parents"][1:] < np.arange(1, 500))
    np.testing.assert_array_equal(t["states"][0], p.start)
