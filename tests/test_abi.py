"""The C-ABI library loads without a GPU and exports every symbol include/hfft.h declares; the
binding refuses to run without a device (no CPU fallback)."""
import os
import re

import numpy as np
import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def hb():
    from paper_1910_07054_b200 import build as hbuild
    hbuild.build()
    from paper_1910_07054_b200 import binding
    return binding


def test_header_symbols_are_exported(hb):
    with open(os.path.join(ROOT, "include", "hfft.h")) as fh:
        src = fh.read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    declared = set(re.findall(r"\b(hfft_[a-z_0-9]+)\s*\(", src))
    assert declared == set(hb.EXPORTS)
    L = hb.lib()
    for name in sorted(declared):
        assert getattr(L, name) is not None
    assert "sm_100a" in hb.version()


def test_info_struct_matches_header(hb):
    with open(os.path.join(ROOT, "include", "hfft.h")) as fh:
        src = fh.read()
    body = re.search(r"typedef struct \{(.*?)\} hfft_info;", src, flags=re.S).group(1)
    body = re.sub(r"/\*.*?\*/", "", body, flags=re.S)
    names = []
    for decl in body.split(";"):
        decl = decl.strip()
        if decl:
            names += [n.strip() for n in decl.split(None, 1)[1].replace("long ", "").split(",")] \
                if not decl.startswith("long long") else [n.strip() for n in decl[len("long long"):].split(",")]
    assert names == [f[0] for f in hb.Info._fields_]


def test_argument_validation_needs_no_device(hb):
    dz = np.array([1.0, 2.0])
    for args, status in [((12, 16, 2, 1.0, 1.0, dz, hb.F32), hb.EUNSUPPORTED),
                         ((16, 16, 2, 0.0, 1.0, dz, hb.F32), hb.EINVAL),
                         ((16, 1, 2, 1.0, 1.0, dz, hb.F32), hb.EINVAL),
                         ((16, 16, 2, 1.0, 1.0, np.array([1.0, np.inf]), hb.F64), hb.EINVAL),
                         ((2048, 16, 2, 1.0, 1.0, dz, hb.F32), hb.EUNSUPPORTED)]:
        with pytest.raises(hb.HfftError) as e:
            hb.plan_create(*args)
        assert e.value.status == status


def test_no_cpu_fallback(hb):
    """Without a CUDA device plan creation must fail loudly (HFFT_ECUDA), never compute on the CPU."""
    import torch
    if torch.cuda.is_available():
        pytest.skip("a device is present")
    with pytest.raises(hb.HfftError) as e:
        hb.plan_create(16, 16, 2, 1.0, 1.0, np.array([1.0, 2.0]), hb.F32)
    assert e.value.status == hb.ECUDA
    with pytest.raises(RuntimeError):
        hb.Plan(16, 16, 2, 1.0, 1.0, np.array([1.0, 2.0]))


def test_product_never_imports_the_oracle():
    pkg = os.path.join(ROOT, "paper_1910_07054_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                with open(os.path.join(dirpath, f)) as fh:
                    txt = fh.read()
                assert "import oracle" not in txt and "from oracle" not in txt and "hfft_oracle" not in txt, f
