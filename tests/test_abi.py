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
