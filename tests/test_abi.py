"""The C-ABI library loads here (no GPU) and exports every symbol include/pic.h declares; calls
that need a device fail loudly instead of falling back to anything."""
import ctypes
import os
import re

import numpy as np
import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def pic():
    from paper_2101_12149_b200 import build
    build.build()
    import paper_2101_12149_b200 as p
    return p


def test_header_symbols_are_all_exported(pic):
    hdr = open(os.path.join(ROOT, "include", "pic.h")).read()
    hdr = re.sub(r"/\*.*?\*/", "", hdr, flags=re.S)
    declared = set(re.findall(r"\b(pic_[a-z_]+)\s*\(", hdr))
    assert declared == set(pic.SYMBOLS)
    L = ctypes.CDLL(pic.LIB_PATH)
    for name in declared:
        assert getattr(L, name) is not None


def test_library_is_sm100a_only(pic):
    import subprocess
    out = subprocess.run(["cuobjdump", "--list-elf", pic.LIB_PATH], capture_output=True, text=True).stdout
    archs = set(re.findall(r"sm_\w+", out))
    assert archs == {"sm_100a"}, archs


def test_default_options(pic):
    o = pic.pic_default_options()
    assert list(o.periodic) == [1, 1, 1] and list(o.tile) == [8, 8, 8]
    assert o.sort_interval == 4 and o.sort_key_mode == 0 and o.deposit_mode == 0
    assert o.pusher == 0 and o.gather_mode == 0 and o.solver == 0


def test_argument_errors_without_device(pic):
    c = 299792458.0
    dx = (1e-6,) * 3
    dt = 0.99 * 1e-6 / (c * 3 ** 0.5)
    with pytest.raises(pic.PicError) as e:
        pic.pic_create((8, 8, 8), dx, dt * 1.05, 1, pic.PIC_F64)
    assert e.value.code == -2          # CFL
    with pytest.raises(pic.PicError) as e:
        pic.pic_create((8, 8, 8), dx, dt, 4, pic.PIC_F64)
    assert e.value.code == -1
    with pytest.raises(pic.PicError) as e:
        pic.pic_create((12, 8, 8), dx, dt, 1, pic.PIC_F64)     # tile 8 does not divide 12
    assert e.value.code == -1
    with pytest.raises(pic.PicError) as e:
        pic.pic_create((2, 8, 8), dx, dt, 1, pic.PIC_F64)
    assert e.value.code == -1


def test_no_cpu_fallback(pic):
    """Without a CUDA device pic_create must fail with PIC_ERR_CUDA (never compute on the host)."""
    try:
        import torch
        if torch.cuda.is_available():
            pytest.skip("a device is present")
    except ImportError:
        pass
    c = 299792458.0
    with pytest.raises(pic.PicError) as e:
        pic.pic_create((8, 8, 8), (1e-6,) * 3, 0.5e-6 / (c * 3 ** 0.5), 1, pic.PIC_F64)
    assert e.value.code == -5
    assert "no CPU fallback" in str(e.value)


def test_null_handle_is_rejected(pic):
    L = pic.lib()
    assert L.pic_step(None, 1) == -1
    assert L.pic_num_particles(None, 0) == -1
    L.pic_destroy(None)


def test_product_does_not_import_oracle():
    pkg = os.path.join(ROOT, "paper_2101_12149_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                src = open(os.path.join(dirpath, f)).read()
                assert "import oracle" not in src and "from oracle" not in src and "liboracle" not in src
                assert "pic_oracle" not in src
    orc = open(os.path.join(ROOT, "oracle", "__init__.py")).read() + open(os.path.join(ROOT, "oracle", "pic_oracle.cpp")).read()
    assert "import paper_2101_12149_b200" not in orc and "libpic" not in orc and "csrc/" not in orc.replace(
        "paper_2101_12149_b200/csrc", "")


def test_ckc_weights_of_the_product_do_what_they_are_built_for(pic):
    """The CUDA side's own CKC weights (pic_ckc_coefficients, host arithmetic, written in the inverse square
    spacings) against what fixes them, with no reference to the oracle's copy: the published cubic-cell
    values 7/12, 1/12, 1/48 (ref [12]); every smoothed difference sums to 1; with c dt = min(dx) the von
    Neumann bound 0 <= (c dt)^2 sum_a S_a sin^2(k_a dx_a/2)/dx_a^2 <= 1 holds for every wave vector and is
    reached; a wave along the finest axis has no dispersion at that time step."""
    import math
    c = 299792458.0
    al, be, ga = pic.pic_ckc_coefficients((1e-6,) * 3)
    assert np.allclose(al, 7 / 12, rtol=1e-15) and np.allclose(ga, 1 / 48, rtol=1e-14)
    assert np.allclose(be[~np.eye(3, dtype=bool)], 1 / 12, rtol=1e-14) and np.all(np.diag(be) == 0)
    for dx in [(1e-6, 1e-6, 1e-6), (1e-6, 0.8e-6, 0.5e-6), (0.1e-6, 0.1e-6, 0.025e-6), (2e-6, 1e-6, 1e-6)]:
        al, be, ga = pic.pic_ckc_coefficients(dx)
        dt = min(dx) / c
        for a in range(3):
            b, cc = (a + 1) % 3, (a + 2) % 3
            assert abs(al[a] + 2 * be[a][b] + 2 * be[a][cc] + 4 * ga[a] - 1) < 1e-15
        th = np.linspace(0, math.pi, 25)
        cx, cy, cz = np.meshgrid(np.cos(th), np.cos(th), np.cos(th), indexing="ij")
        sx, sy, sz = np.meshgrid(np.sin(th / 2) ** 2, np.sin(th / 2) ** 2, np.sin(th / 2) ** 2, indexing="ij")
        cs, s2 = (cx, cy, cz), (sx, sy, sz)
        tot = 0.0
        for a in range(3):
            b, cc = (a + 1) % 3, (a + 2) % 3
            S = al[a] + 2 * be[a][b] * cs[b] + 2 * be[a][cc] * cs[cc] + 4 * ga[a] * cs[b] * cs[cc]
            tot = tot + S * s2[a] / dx[a] ** 2
        tot = tot * (c * dt) ** 2
        assert tot.min() > -1e-14 and tot.max() <= 1 + 1e-12 and tot.max() > 0.999
        # along the finest axis alone: S = 1, so sin^2(omega dt/2) = sin^2(k dx/2), i.e. omega = c k
        a = int(np.argmin(dx))
        b, cc = (a + 1) % 3, (a + 2) % 3
        assert abs(al[a] + 2 * be[a][b] + 2 * be[a][cc] + 4 * ga[a] - 1) < 1e-15
    with pytest.raises(pic.PicError):
        pic.pic_ckc_coefficients((1e-6, 0.0, 1e-6))
