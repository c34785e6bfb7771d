"""CPU-side checks of the boundary: the C-ABI library loads, exports every symbol include/tm.h declares, and
its host-only logic behaves (no device compute here)."""
import ctypes
import os
import re

import numpy as np
import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def libtm():
    from paper_2107_09879_b200 import build, libtm as m
    build.build()
    return m


def test_exports_match_header(libtm):
    hdr = open(os.path.join(ROOT, "include", "tm.h")).read()
    hdr = re.sub(r"/\*.*?\*/", "", hdr, flags=re.S)
    declared = set(re.findall(r"\b(tm_[A-Za-z_0-9]+)\s*\(", hdr))
    assert declared == set(libtm.EXPORTS)
    lib = libtm.lib()
    for name in declared:
        assert hasattr(lib, name), name


def test_num_modes_and_enums(libtm):
    lib = libtm.lib()
    assert [lib.tm_num_modes(l) for l in (1, 2, 3, 6)] == [6, 16, 30, 96]
    hdr = open(os.path.join(ROOT, "include", "tm.h")).read()
    for name in ("TM_FP64", "TM_FP32", "TM_OK", "TM_NOT_CONVERGED", "TM_E_INVALID", "TM_E_OVERLAP", "TM_E_STATE",
                 "TM_E_CUDA", "TM_E_NOMEM", "TM_INC_PLANE", "TM_INC_GAUSS", "TM_INC_COEFFS", "TM_INC_JINC", "TM_FIELD_E_SCA",
                 "TM_FIELD_H_SCA", "TM_FIELD_E_INC", "TM_MIXED", "TM_KERNEL_AUTO", "TM_KERNEL_GENERAL", "TM_KERNEL_COPLANAR", "TM_KERNEL_SYM3D", "TM_KERNEL_ROT3D", "TM_PEAK_FP64_TENSOR"):
        m = re.search(name + r"\s*=\s*(-?\d+)", hdr)
        assert m and int(m.group(1)) == getattr(libtm, name), name


def test_struct_layouts(libtm, tmp_path):
    """The ctypes mirrors have the layout the C compiler gives include/tm.h (sizes and the offset of every field)."""
    import subprocess
    pairs = [("tm_c64", libtm.c64), ("tm_plane_desc", libtm.PlaneDesc), ("tm_gauss_desc", libtm.GaussDesc),
             ("tm_jinc_desc", libtm.JincDesc), ("tm_coeffs_desc", libtm.CoeffsDesc), ("tm_solve_opts", libtm.SolveOpts),
             ("tm_solve_info", libtm.SolveInfo)]
    lines = ['#include <stddef.h>', '#include <stdio.h>', '#include "tm.h"', "int main(void) {"]
    for cname, ct in pairs:
        lines.append(f'  printf("{cname} %zu\\n", sizeof({cname}));')
        for fname, _ in ct._fields_:
            lines.append(f'  printf("{cname}.{fname} %zu\\n", offsetof({cname}, {fname}));')
    lines += ["  return 0;", "}"]
    src = tmp_path / "layout.c"
    src.write_text("\n".join(lines))
    exe = tmp_path / "layout"
    subprocess.run(["gcc", "-std=c99", "-I", os.path.join(ROOT, "include"), str(src), "-o", str(exe)], check=True)
    got = dict(l.split() for l in subprocess.run([str(exe)], check=True, capture_output=True, text=True).stdout.splitlines())
    for cname, ct in pairs:
        assert int(got[cname]) == ctypes.sizeof(ct), cname
        for fname, _ in ct._fields_:
            assert int(got[f"{cname}.{fname}"]) == getattr(ct, fname).offset, f"{cname}.{fname}"
    assert ctypes.sizeof(libtm.SolveOpts) == 24 and libtm.SolveOpts.warm_start.offset == 16


def test_mie_host_helper_lossless_and_argument_checks(libtm):
    t = libtm.mie_tmatrix(3, 2 * np.pi, 0.2, 4.0)
    assert t.shape == (30,)
    assert np.abs(np.abs(1 + 2 * t) - 1).max() < 1e-13          # lossless sphere: |S| = 1
    assert np.allclose(t[0:3], t[0]) and np.allclose(t[15:18], t[15])   # independent of m
    with pytest.raises(libtm.TmError):
        libtm.mie_tmatrix(0, 2 * np.pi, 0.2, 4.0)
    with pytest.raises(libtm.TmError):
        libtm.mie_tmatrix(3, 2 * np.pi, -1.0, 4.0)


def test_create_validates_before_touching_the_device(libtm):
    pos = np.zeros((2, 3)); pos[1, 0] = 1.0
    with pytest.raises(libtm.TmError) as e:
        libtm.Solver(pos, 0, 2 * np.pi)
    assert e.value.code == libtm.TM_E_INVALID
    with pytest.raises(libtm.TmError) as e:
        libtm.Solver(pos, 2, 2 * np.pi, win_ptr=[0, 1, 3])
    assert e.value.code == libtm.TM_E_INVALID


def test_no_cpu_fallback(libtm):
    """Without a CUDA device the product refuses to run (TM_E_CUDA); it never routes through the oracle."""
    import torch
    if torch.cuda.is_available():
        pytest.skip("a GPU is present")
    pos = np.zeros((2, 3)); pos[1, 0] = 1.0
    with pytest.raises(libtm.TmError) as e:
        libtm.Solver(pos, 2, 2 * np.pi)
    assert e.value.code == libtm.TM_E_CUDA
    src = open(os.path.join(ROOT, "paper_2107_09879_b200", "libtm.py")).read()
    assert "oracle" not in src.replace("no CPU fallback", "")
