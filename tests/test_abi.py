"""CPU-side checks of the C-ABI library (no compute calls): it loads, exports every symbol include/fsw.h declares,
its struct layouts match the ctypes binding, and its host logic (rig / plane-set validation and precompute, S0 of
SURVEY.md 8(a)) gives the closed-form values the conventions fix (and agrees with the oracle's O2/O3)."""
import ctypes
import os
import re
import subprocess
import sys
import tempfile

import numpy as np
import pytest

import oracle
import synth
import paper_1809_06132_b200 as fsw
from paper_1809_06132_b200 import binding

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
HEADER = os.path.join(ROOT, "include", "fsw.h")


def _declared_functions():
    text = open(HEADER).read()
    text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)
    return sorted(set(re.findall(r"\b(fsw_[a-z0-9_]+)\s*\(", text)))


def test_library_exports_every_declared_symbol():
    lib = fsw.load_library()
    names = _declared_functions()
    assert len(names) >= 18
    for name in names:
        assert hasattr(lib, name), name
    from paper_1809_06132_b200.tsdf import TSDF_EXPORTS
    assert sorted(binding.EXPORTS + TSDF_EXPORTS) == names
    assert fsw.version() == (0, 3)


def test_struct_layouts_match_header():
    """sizeof / offsetof of every ABI struct, as compiled by gcc from include/fsw.h, equal the ctypes mirror."""
    structs = {"fsw_camera": binding.CCamera, "fsw_plane_family": binding.CFamily, "fsw_rect": binding.CRect,
               "fsw_sweep_params": binding.CParams, "fsw_image": binding.CImage, "fsw_depth_out": binding.CDepthOut,
               "fsw_counters": binding.CCounters, "fsw_schedule_plan": binding.CSchedulePlan}
    from paper_1809_06132_b200 import tsdf
    structs.update({"fsw_tsdf_params": tsdf.CTsdfParams, "fsw_tsdf_stats": tsdf.CTsdfStats})
    lines = ['#include <stdio.h>', '#include <stddef.h>', '#include "fsw.h"', 'int main(void){']
    for cname, cls in structs.items():
        lines.append('printf("%s %%zu\\n", sizeof(%s));' % (cname, cname))
        for fname, _ in cls._fields_:
            lines.append('printf("%s.%s %%zu\\n", offsetof(%s, %s));' % (cname, fname, cname, fname))
    lines.append("return 0;}")
    with tempfile.TemporaryDirectory() as d:
        src, exe = os.path.join(d, "t.c"), os.path.join(d, "t")
        open(src, "w").write("\n".join(lines))
        subprocess.check_call(["gcc", "-I", os.path.join(ROOT, "include"), src, "-o", exe])
        got = dict(line.split() for line in subprocess.check_output([exe], text=True).splitlines())
    for cname, cls in structs.items():
        assert int(got[cname]) == ctypes.sizeof(cls), cname
        for fname, _ in cls._fields_:
            assert int(got["%s.%s" % (cname, fname)]) == getattr(cls, fname).offset, (cname, fname)


def _yaw(deg):
    """Closed form of reading Q5: rig -> camera rotation of a camera yawed by `deg` about +y (down); a positive yaw
    turns the optical axis towards +x, so the rig point (sin, 0, cos) lies on the optical axis."""
    a = np.radians(deg)
    return np.array([[np.cos(a), 0.0, -np.sin(a)], [0.0, 1.0, 0.0], [np.sin(a), 0.0, np.cos(a)]])


def test_rig_validation_and_relative_pose():
    cfg = synth.make_config(2)   # reference at the origin; views at x = -+0.4 m, yawed by -+10 degrees
    rig = fsw.Rig(cfg["cams"], 0)
    for c, (centre, yaw) in ((1, ((-0.4, 0.0, 0.0), -10.0)), (2, ((0.4, 0.0, 0.0), 10.0))):
        R, T = rig.relative_pose(c)
        # closed form: the reference frame is the rig frame, so X_v = R_y (X - C): R = R_y, T = -R_y C
        assert np.allclose(R, _yaw(yaw), atol=1e-15) and np.allclose(T, -_yaw(yaw) @ np.array(centre), atol=1e-15)
        assert np.allclose(R @ np.array([np.sin(np.radians(yaw)), 0.0, np.cos(np.radians(yaw))]), (0, 0, 1), atol=1e-15)
        Ro, To = oracle.relative_pose(cfg["cams"][0], cfg["cams"][c])
        assert np.allclose(R, Ro, atol=1e-15) and np.allclose(T, To, atol=1e-15)
    # between two yawed cameras: the rotation is the difference of the yaws, and the reference's centre maps to T
    rig12 = fsw.Rig(cfg["cams"], 1)
    R, T = rig12.relative_pose(2)
    assert np.allclose(R, _yaw(20.0), atol=1e-15)
    assert np.allclose(T, _yaw(10.0) @ (np.array([-0.4, 0, 0]) - np.array([0.4, 0, 0])), atol=1e-15)
    Rb, Tb = fsw.Rig(cfg["cams"], 2).relative_pose(1)    # the inverse pose
    assert np.allclose(Rb @ R, np.eye(3), atol=1e-15) and np.allclose(Rb @ T + Tb, 0.0, atol=1e-15)
    R0, T0 = rig.relative_pose(0)
    assert np.array_equal(R0, np.eye(3)) and np.array_equal(T0, np.zeros(3))
    # a sub-rig keeps the reference and the poses of the cameras it lists
    sub = rig.subset([2, 0])
    assert (sub.n_cams, sub.ref_index) == (2, 1)
    assert np.array_equal(sub.relative_pose(0)[0], rig.relative_pose(2)[0]) and np.array_equal(sub.relative_pose(0)[1], rig.relative_pose(2)[1])
    for bad_subset in ([1, 2], [0], [0, 0], [0, 5]):
        with pytest.raises(fsw.FswError) as ei:
            rig.subset(bad_subset)
        assert ei.value.code == fsw.binding.E_INVALID_ARG
    # ground normal: rig "down" expressed in a yawed reference camera stays "down"
    rig2 = fsw.Rig(cfg["cams"], 1)
    assert np.allclose(rig2.ground_normal_in_ref((0, 2.0, 0)), (0, 1, 0), atol=1e-15)
    good = cfg["cams"][0]

    def bad(**kw):
        c = dict(good)
        c.update(kw)
        return c

    cases = [
        ([good], 0, fsw.binding.E_INVALID_ARG),                      # a rig needs two cameras
        ([good, good], 2, fsw.binding.E_INVALID_ARG),                # reference index out of range
        ([good, bad(fx=0.0)], 0, fsw.binding.E_CONFIG),
        ([good, bad(cx=-5.0)], 0, fsw.binding.E_CONFIG),             # principal point outside the image
        ([good, bad(xi=3.5)], 0, fsw.binding.E_CONFIG),
        ([good, bad(fov_max_deg=0.0)], 0, fsw.binding.E_CONFIG),
        ([good, bad(R=np.eye(3) * 1.01)], 0, fsw.binding.E_CONFIG),  # not orthonormal
        ([good, bad(R=np.diag([1.0, 1.0, -1.0]))], 0, fsw.binding.E_CONFIG),  # reflection
        ([good, bad(k1=-0.5)], 0, fsw.binding.E_CONFIG),             # distortion folds over inside the FOV
    ]
    for cams, ref, code in cases:
        with pytest.raises(fsw.FswError) as ei:
            fsw.Rig(cams, ref)
        assert ei.value.code == code, (ei.value, code)
    with pytest.raises(fsw.FswError):
        fsw.Rig([good] * 9, 0)


def test_planeset_table_matches_oracle_and_validation():
    # the values SURVEY.md 8(c) prints for C1 (tests/golden/survey_spot_values.txt): 32 planes uniform in 1/d over
    # 0.5..50 m
    from conftest import read_golden
    g = read_golden(os.path.join(ROOT, "tests", "golden", "survey_spot_values.txt"))["c1_planes"]
    s, d, f = fsw.PlaneSet(synth.make_config(1)["families"]).table()
    assert abs((s[0] - s[1]) - g[0]) < 5e-8 and abs(d[0] - g[1]) < 1e-12 and abs(d[27] - g[2]) < 5e-6
    assert abs(d[28] - g[3]) < 5e-6 and abs(d[31] - g[4]) < 1e-9
    # closed form: k-th of n planes is the point k/(n-1) of the way in the spacing variable
    s, d, f = fsw.PlaneSet([synth.family((0, 0, 1), 5, 2.0, 10.0, "linear"), synth.family((0, 1, 0), 3, 1.0, 4.0, "inverse")]).table()
    assert np.allclose(s, [2, 4, 6, 8, 10, 1.0, 0.625, 0.25], atol=1e-15) and np.allclose(d[5:], [1.0, 1.6, 4.0], atol=1e-15)
    assert list(f) == [0] * 5 + [1] * 3
    for idx in (1, 3, 5):
        fams = synth.make_config(idx)["families"]
        ps = fsw.PlaneSet(fams)
        s, d, f = ps.table()
        so, do, fo, _ = oracle.plane_table(fams)
        assert ps.n_planes == len(so)
        assert np.allclose(s, so, rtol=0, atol=1e-15) and np.allclose(d, do, rtol=1e-15) and np.array_equal(f, fo)
    one = synth.family((0, 0, 2.0), 1, 3.0, 7.0, "inverse")
    assert np.allclose(fsw.PlaneSet([one]).table()[1], [3.0])
    E = fsw.binding
    cases = [
        ([], E.E_INVALID_ARG),
        ([synth.family((0, 0, 1), 0, 1.0, 2.0, "inverse")], E.E_CONFIG),
        ([synth.family((0, 0, 1), 4, -1.0, 2.0, "inverse")], E.E_CONFIG),
        ([synth.family((0, 0, 0), 4, 1.0, 2.0, "inverse")], E.E_CONFIG),
        ([synth.family((0, 0, 1), 600, 1.0, 2.0, "inverse")] * 2, E.E_CONFIG),   # more than FSW_MAX_PLANES
        ([dict(synth.family((0, 0, 1), 4, 1.0, 2.0, "inverse"), spacing=7)], E.E_INVALID_ARG),
    ]
    for fams, code in cases:
        with pytest.raises(fsw.FswError) as ei:
            fsw.PlaneSet(fams)
        assert ei.value.code == code, (ei.value, code)


def test_no_cpu_fallback():
    """Without a CUDA device the product path fails loudly instead of computing on the CPU."""
    import torch
    if torch.cuda.is_available():
        pytest.skip("a CUDA device is present")
    rig = fsw.Rig(synth.make_config(1)["cams"], 0)
    with pytest.raises(fsw.FswError) as ei:
        fsw.Context(rig, 0)
    assert ei.value.code == fsw.binding.E_CUDA


def test_product_does_not_import_oracle():
    """The CUDA path and the oracle share no code: nothing under paper_1809_06132_b200/ mentions oracle/."""
    pkg = os.path.join(ROOT, "paper_1809_06132_b200")
    for dirpath, _, files in os.walk(pkg):
        if "build" in os.path.relpath(dirpath, pkg).split(os.sep)[:1]:
            continue
        for fn in files:
            if fn.endswith((".py", ".cu", ".cuh", ".h")):
                text = open(os.path.join(dirpath, fn)).read()
                assert "import oracle" not in text and "from oracle" not in text and "fsw_oracle" not in text, fn
    code = "import sys; sys.path.insert(0, %r); import paper_1809_06132_b200; assert 'oracle' not in sys.modules" % ROOT
    subprocess.check_call([sys.executable, "-c", code])
