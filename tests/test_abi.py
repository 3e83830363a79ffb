"""The C-ABI library loads and exports every symbol include/satsplat.h declares (no compute calls: no GPU here),
the host-side camera helper agrees with the oracle's Eq. 16, and the product package never imports the oracle."""
import ctypes
import os
import re

import numpy as np

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _declared():
    src = open(os.path.join(ROOT, "include", "satsplat.h")).read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    return sorted(set(re.findall(r"\b(satsplat_[a-z_0-9]+)\s*\(", src)))


def test_library_exports_every_declared_symbol():
    import paper_2606_28581_b200 as P
    P.build()
    lib = ctypes.CDLL(os.path.join(ROOT, "paper_2606_28581_b200", "libsatsplat.so"))
    names = _declared()
    assert len(names) >= 17 and "satsplat_preprocess" in names and "satsplat_render_backward" in names
    for n in names:
        assert hasattr(lib, n), n
    assert b"sm_100a" in ctypes.c_char_p(ctypes.cast(lib.satsplat_version, ctypes.CFUNCTYPE(ctypes.c_char_p))()).value


def test_error_paths_without_gpu():
    import paper_2606_28581_b200 as P
    L = P.lib()
    assert L.satsplat_preprocess(None, None, 0, None, None, None, None, None, None) == P.E_INVALID
    assert b"NULL" in L.satsplat_last_error(None)
    out = ctypes.c_void_p()
    assert L.satsplat_create(ctypes.byref(out), 0, -1, 16, 16, 10) == P.E_INVALID
    assert L.satsplat_create(ctypes.byref(out), 0, 10, 0, 16, 10) == P.E_INVALID
    L.satsplat_destroy(None)


def test_sun_camera_helper_matches_oracle(orc):
    import paper_2606_28581_b200 as P
    import satsplat_scenes as S
    rng = np.random.default_rng(7)
    for _ in range(10):
        F, d = S.affine_camera(0.4, np.radians(rng.uniform(0, 35)), rng.uniform(0, 6.28), 512, 512, (64, 64, 0))
        dF = rng.normal(0, 1e-3, 8).astype(np.float32)
        cam = P.Camera.make(512, 512, F, dF, d, b_z=60.0, z_bg=70.0)
        az, el = rng.uniform(0, 6.28), np.radians(rng.uniform(25, 75))
        vp = np.array([0.8, 0.8, 100.0, 90.0], np.float32)
        sun, rep = P.sun_camera(cam, az, el, 1024, 1024, vp)
        Fp = (F + dF).astype(np.float64)
        F_ref, rep_ref = orc.sun_camera(Fp, np.float32(az), np.float32(el), vp)
        np.testing.assert_allclose(np.array(sun.F[:]), F_ref, rtol=1e-6, atol=1e-5)
        np.testing.assert_allclose(np.array(rep), rep_ref, rtol=1e-6, atol=1e-5)
        assert sun.b_z == cam.b_z and sun.width == 1024
    bad = P.Camera.make(8, 8, [0] * 8)
    try:
        P.sun_camera(bad, 0.0, 1.0, 8, 8, [1, 1, 0, 0])
        assert False
    except P.SatsplatError as e:
        assert e.code == P.E_INVALID


def test_product_does_not_touch_the_oracle():
    pkg = os.path.join(ROOT, "paper_2606_28581_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                txt = open(os.path.join(dirpath, f)).read()
                assert "import oracle" not in txt and "from oracle" not in txt and "satsplat_oracle" not in txt, f
    otxt = open(os.path.join(ROOT, "oracle", "oracle.py")).read() + open(os.path.join(ROOT, "oracle", "satsplat_oracle.cpp")).read()
    assert "paper_2606_28581_b200 import" not in otxt and "import paper_2606_28581_b200" not in otxt
    assert "#include \"../paper" not in otxt and "satsplat.h" not in otxt
