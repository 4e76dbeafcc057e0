"""C-ABI checks that need no GPU: the library builds, loads, exports every symbol include/omerf.h
declares, validates arguments, and fails loudly (never falls back to a CPU path) without a device."""
import ctypes as C
import os
import re

import numpy as np
import pytest

import synth

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def omerf():
    from paper_2404_09531_b200 import build as b
    b.build()
    import paper_2404_09531_b200 as m
    return m


def test_every_declared_symbol_is_exported(omerf):
    hdr = open(os.path.join(ROOT, "include", "omerf.h")).read()
    hdr = re.sub(r"/\*.*?\*/", "", hdr, flags=re.S)
    declared = set(re.findall(r"\b(omerf_[a-z_]+)\s*\(", hdr))
    assert declared == set(omerf.EXPORTS)
    L = omerf.load_library()
    for name in declared:
        assert getattr(L, name) is not None
    assert b"sm_100a" in L.omerf_version()


def test_range_checked_flavour_builds_and_exports_the_same_symbols(omerf):
    """libomerf_checked.so (-DOMERF_CHECKED, tests/test_gpu_checked.py): same C-ABI as the shipped library"""
    from paper_2404_09531_b200 import build as b
    L = C.CDLL(b.build(checked=True))
    for name in omerf.EXPORTS:
        assert getattr(L, name) is not None
    L.omerf_check_errors.restype = C.c_uint32
    assert omerf.load_library().omerf_check_errors() == 0          # the shipped library has no checks: always 0


def test_struct_layout_matches_header(omerf, tmp_path):
    """ctypes mirrors vs the real header, through gcc's offsetof/sizeof."""
    import subprocess
    from paper_2404_09531_b200.binding import SceneDesc, SceneInfo
    fields = [n for n, _ in SceneDesc._fields_]
    src = tmp_path / "layout.c"
    lines = ['#include <stdio.h>', '#include <stddef.h>', f'#include "{ROOT}/include/omerf.h"', 'int main(void){',
             'printf("%zu %zu %zu\\n", sizeof(omerf_scene_desc), sizeof(omerf_scene_info), sizeof(omerf_camera));']
    lines += [f'printf("%zu\\n", offsetof(omerf_scene_desc, {f}));' for f in fields]
    lines += ['return 0;}']
    src.write_text("\n".join(lines))
    exe = tmp_path / "layout"
    subprocess.check_call(["gcc", "-o", str(exe), str(src)])
    out = subprocess.check_output([str(exe)]).decode().split()
    assert [int(x) for x in out[:3]] == [C.sizeof(SceneDesc), C.sizeof(SceneInfo), 64]
    assert [int(x) for x in out[3:]] == [getattr(SceneDesc, f).offset for f in fields]


def test_invalid_arguments_are_rejected_before_touching_cuda(omerf):
    from paper_2404_09531_b200.binding import make_desc
    L = omerf.load_library()
    sc = synth.custom_scene()
    out = C.c_void_p()
    assert L.omerf_scene_create(None, C.byref(out)) == -1
    for mutate, word in [
        (lambda d: setattr(d, "step", 0.0), "step"),
        (lambda d: setattr(d, "t_stop", 1.5), "t_stop"),
        (lambda d: setattr(d, "mlp_in", 33), "MLP"),
        (lambda d: setattr(d, "h_lo", None), "height"),
        (lambda d: d.grid_n.__setitem__(0, 0), "grid_n"),
        (lambda d: setattr(d, "sampler", 7), "sampler"),
        (lambda d: d.box.__setitem__(2, -1.0), "box"),
    ]:
        d, keep = make_desc(sc)
        mutate(d)
        assert L.omerf_scene_create(C.byref(d), C.byref(out)) == -1
        assert word in L.omerf_last_error().decode()
        assert not out.value
    d, keep = make_desc(sc, sampler=1)          # grid sampler needs occ_n
    assert L.omerf_scene_create(C.byref(d), C.byref(out)) == -1
    # 8(f) options that are defined by the slab need the occupancy-plane sampler: the grid sampler's voxels are a superset
    sg = synth.custom_scene(occ_n=(8, 8, 8))
    for kw, word in (({"grid_block": 4}, "grid_block"), ({"soft_eps": 0.5}, "soft_eps")):
        d, keep = make_desc(sg, sampler=1, **kw)
        assert L.omerf_scene_create(C.byref(d), C.byref(out)) == -1
        assert word in L.omerf_last_error().decode() and not out.value
    assert L.omerf_render(None, None, 1, 4, 4, None, None, None) == -1
    assert L.omerf_render_host(None, None, 1, 4, 4, None, None, None) == -1
    L.omerf_scene_destroy(None)                  # no-op


def test_no_cpu_fallback_without_a_device(omerf):
    import torch
    if torch.cuda.is_available():
        pytest.skip("a GPU is present")
    with pytest.raises(omerf.OmerfError):
        omerf.scene_create(synth.custom_scene())
    # and at the C level: a valid description fails with a CUDA error code, not a silent CPU path
    from paper_2404_09531_b200.binding import make_desc
    L = omerf.load_library()
    d, keep = make_desc(synth.custom_scene())
    out = C.c_void_p()
    rc = L.omerf_scene_create(C.byref(d), C.byref(out))
    assert rc in (-2, -3) and not out.value
    assert b"CUDA" in L.omerf_last_error()


def test_product_package_does_not_import_the_oracle():
    pkg = os.path.join(ROOT, "paper_2404_09531_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            path = os.path.join(dirpath, f)
            if f.endswith(".py"):
                src = open(path).read()
                assert not re.search(r"^\s*(import|from)\s+oracle\b", src, flags=re.M), f
                assert "liboracle" not in src and "omerf_oracle" not in src and '"oracle"' not in src, f
            elif f.endswith((".cu", ".cuh", ".h")):
                src = open(path).read()
                assert not re.search(r"#\s*include[^\n]*oracle", src), f
    for f in os.listdir(os.path.join(ROOT, "oracle")):
        if f.endswith((".py", ".c", ".h")):
            src = open(os.path.join(ROOT, "oracle", f)).read()
            assert "paper_2404_09531_b200" not in src.replace("(paper_2404_09531_b200/csrc", "").replace(
                "(paper_2404_09531_b200)", "")
            assert not re.search(r"#\s*include[^\n]*omerf\.h", src)
