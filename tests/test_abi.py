"""The C-ABI library loads and exports every symbol include/*.h declares (no compute; runs without a GPU)."""
import ctypes
import os
import re

import numpy as np
import pytest

import paper_1602_06645_b200 as vf

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def declared_symbols():
    names = set()
    for header in sorted(os.listdir(os.path.join(ROOT, "include"))):
        src = open(os.path.join(ROOT, "include", header)).read()
        src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
        names |= set(re.findall(r"\b(vol_[a-z_]+)\s*\(", src))
    return sorted(names)


def test_header_symbols_are_exported():
    L = vf.lib()
    names = declared_symbols()
    assert set(names) == set(vf.EXPORTS)
    for n in names:
        assert getattr(L, n) is not None


def test_struct_layouts_match_header(tmp_path):
    """The header is plain C, and the ctypes mirrors have the sizes / offsets gcc gives the ABI structs."""
    import subprocess
    src = tmp_path / "sz.c"
    src.write_text('#include <stdio.h>\n#include <stddef.h>\n#include "volfusion.h"\n'
                   'int main(void){printf("%zu %zu %zu %zu %zu %zu\\n", sizeof(vol_opts_t), sizeof(vol_info_t), sizeof(vol_stats_t),'
                   ' offsetof(vol_info_t, geo_bytes), offsetof(vol_info_t, col_dev), offsetof(vol_stats_t, tiles_total));return 0;}\n')
    exe = tmp_path / "sz"
    subprocess.run(["gcc", "-std=c99", "-Wall", "-Werror", "-I", os.path.join(ROOT, "include"), str(src), "-o", str(exe)], check=True)
    got = [int(x) for x in subprocess.run([str(exe)], check=True, capture_output=True, text=True).stdout.split()]
    assert got == [ctypes.sizeof(vf.VolOpts), ctypes.sizeof(vf.VolInfo), ctypes.sizeof(vf.VolStats),
                   vf.VolInfo.geo_bytes.offset, vf.VolInfo.col_dev.offset, vf.VolStats.tiles_total.offset]


def test_argument_validation_precedes_any_cuda_call():
    L = vf.lib()
    h = ctypes.c_void_p()
    org = (ctypes.c_float * 3)(0, 0, 0)
    bad = [((0, 8, 8), 2, 1.0, 0.1, 128), ((8, -3, 8), 2, 1.0, 0.1, 128), ((8, 8, 8), 0, 1.0, 0.1, 128),
           ((8, 8, 8), 5, 1.0, 0.1, 128), ((8, 8, 8), 2, -1.0, 0.1, 128), ((8, 8, 8), 2, 1.0, 0.0, 128),
           ((8, 8, 8), 2, 1.0, 0.1, 0), ((8, 8, 8), 2, 1.0, 0.1, 513)]
    for dims, r, ext, mu, wmax in bad:
        d = (ctypes.c_int32 * 3)(*dims)
        assert L.vol_create(ctypes.byref(h), d, r, org, ext, mu, wmax, None) == vf.VOL_E_ARG
        assert not h
    assert L.vol_create(None, None, 2, org, 1.0, 0.1, 128, None) == vf.VOL_E_ARG
    assert L.vol_strerror(vf.VOL_E_ARG) == b"invalid argument"
    assert L.vol_integrate(None, None, 1, 1, None, 1, 1, None, None, None, None, None) == vf.VOL_E_ARG
    fe = ctypes.c_void_p()
    for w, h, levels in ((0, 8, 1), (8, 8, 0), (8, 8, 7), (12, 8, 4), (8, 6, 3)):
        assert L.vol_frontend_create(ctypes.byref(fe), w, h, levels, None) == vf.VOL_E_ARG and not fe
    assert L.vol_frontend_measure(None, None, None, None) == vf.VOL_E_ARG


def test_no_cpu_fallback_without_a_gpu():
    import torch
    if torch.cuda.is_available():
        pytest.skip("a GPU is present")
    with pytest.raises(vf.VolError) as e:
        vf.Volume((8, 8, 8), 2, (0, 0, 0), 1.0, 0.1, 128)
    assert e.value.code == vf.VOL_E_CUDA


def test_parity_harness_describes_a_mismatch():
    """tests/parity_util.describe_mismatches (SURVEY 8(c) diagnostics): a word changed by hand is reported with its voxel
    index, both words' fields and where the voxel stands relative to the decisions that gate its update."""
    import numpy as np
    import oracle
    import synth
    from parity_util import describe_mismatches
    c = synth.config(1).scaled(32, 2)
    o = oracle.RefVolume(c.dims_geo, c.r, c.origin, c.extent, c.mu, c.w_max)
    depth, rgb, T = synth.frame(c, 0)
    o.integrate(depth, rgb, T, c.K_depth, c.K_rgb, c.T_depth_rgb)
    geo, col = o.geo.copy(), o.col.copy()
    assert describe_mismatches(geo, o.geo, col, o.col, o) == ""
    gi, ci = np.flatnonzero(geo)[100], np.flatnonzero(col)[50]
    geo.reshape(-1)[gi] ^= 1
    col.reshape(-1)[ci] ^= 0x100
    txt = describe_mismatches(geo, o.geo, col, o.col, o, (c, depth, T))
    assert "geometry: 1 words differ" in txt and "colour: 1 words differ" in txt
    assert "sdf + mu" in txt and "d^2 - sigma^2" in txt and "(u, v)" in txt and "oracle q =" in txt
