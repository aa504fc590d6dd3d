"""CPU-side checks of the boundary: libxf.so builds, loads and exports every symbol include/xf.h declares; argument
errors are reported before any CUDA work; without a device xf_create fails loudly (no CPU fallback)."""
import ctypes as C
import re
from pathlib import Path

import numpy as np
import pytest

ROOT = Path(__file__).resolve().parent.parent


@pytest.fixture(scope="module")
def xf():
    from paper_2403_05910_b200 import build, xf as mod

    build.build()
    return mod


def declared_symbols():
    text = (ROOT / "include" / "xf.h").read_text()
    text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)
    return sorted(set(re.findall(r"\b(xf_[a-z0-9_]+)\s*\(", text)))


def test_library_exports_every_declared_symbol(xf):
    names = declared_symbols()
    assert set(names) == set(xf.ABI_SYMBOLS)
    L = C.CDLL(str(xf.LIB_PATH))
    for n in names:
        assert hasattr(L, n), n


def test_config_struct_matches_header_order(xf):
    text = (ROOT / "include" / "xf.h").read_text()
    body = re.search(r"typedef struct \{(.*?)\} xf_config;", text, flags=re.S).group(1)
    body = re.sub(r"/\*.*?\*/", "", body, flags=re.S)
    fields = []
    for decl in body.split(";"):
        decl = decl.strip()
        if not decl:
            continue
        for name in decl.split(","):
            fields.append(re.sub(r"\[.*\]", "", name.strip().split()[-1].lstrip("*")))
    assert fields == [f[0] for f in xf.XfConfig._fields_]


def _cfg(xf, **over):
    kw = dict(nx=16, ny=1, nz=1, dx=0.1, dy=1.0, dz=1.0, W=[28.0, 4.0],
              nasa7=np.array([[3.5, 0, 0, 0, 0, 0, 0], [2.5, 0, 0, 0, 0, 0, 0]], dtype=float), Ru=1.0, Tlo=0.0, Thi=1e300)
    kw.update(over)
    return kw


def test_invalid_arguments_are_rejected_before_cuda(xf):
    for bad in (dict(nx=0), dict(nx=2), dict(dx=0.0), dict(Ru=-1.0), dict(Thi=-1.0), dict(bc=(0, 1, 0, 0, 0, 0)),
                dict(bc=(3, 1, 0, 0, 0, 0)), dict(bc=(7, 7, 0, 0, 0, 0)), dict(nx=1)):
        with pytest.raises(xf.XfError) as e:
            xf.Context(**_cfg(xf, **bad))
        assert e.value.code == xf.XF_EINVAL, bad
    assert xf.lib().xf_create(None, None) == xf.XF_EINVAL
    assert xf.lib().xf_destroy(None) == xf.XF_EINVAL
    assert xf.lib().xf_status(None, None) == xf.XF_EINVAL
    assert "invalid" in xf.strerror(xf.XF_EINVAL)


def test_no_device_means_loud_failure_not_a_fallback(xf):
    import torch

    if torch.cuda.is_available():
        pytest.skip("a CUDA device is present")
    with pytest.raises(xf.XfError) as e:
        xf.Context(**_cfg(xf))
    assert e.value.code == xf.XF_ECUDA


def test_product_never_imports_the_oracle():
    pkg = ROOT / "paper_2403_05910_b200"
    for f in list(pkg.rglob("*.py")) + list(pkg.rglob("*.cu")) + list(pkg.rglob("*.cuh")):
        s = f.read_text()
        assert "oracle" not in s.replace("oracle/", "").replace("the oracle", "").replace("oracle tests", "") or \
            not re.search(r"^\s*(import|from)\s+oracle|xf_oracle\.h|libxf_oracle", s, flags=re.M), f
    for f in (ROOT / "oracle").glob("*"):
        if f.suffix in (".py", ".c", ".h"):
            assert not re.search(r"^\s*(import|from)\s+paper_2403_05910_b200|include\s*\"xf\.h\"", f.read_text(), flags=re.M), f
