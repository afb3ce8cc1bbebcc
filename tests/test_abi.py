"""CPU-side checks of the boundary: the C-ABI library loads and exports every symbol include/rt.h declares."""
import os
import re

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _declared():
    src = open(os.path.join(ROOT, "include", "rt.h")).read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    return sorted(set(re.findall(r"\b(rt_[a-z_0-9]+)\s*\(", src)))


def test_header_declares_the_north_star_calls():
    names = _declared()
    for n in ("rt_init", "rt_transport", "rt_angular_flux", "rt_source_implicit", "rt_moments", "rt_step"):
        assert n in names


def test_library_builds_loads_and_exports_every_symbol():
    from paper_2508_15532_b200 import build, rt
    build.build()
    lib = rt.load_library()
    for n in _declared():
        assert hasattr(lib, n), n
    assert sorted(rt.SYMBOLS) == _declared()
    assert lib.rt_strerror(0) == b"ok" and lib.rt_strerror(-1) == b"invalid argument"
    # argument validation happens before any CUDA call
    assert lib.rt_ndir(None) == -1 and lib.rt_free(None) == -1


def test_no_fallback_without_gpu():
    import torch
    from paper_2508_15532_b200 import rt
    if torch.cuda.is_available():
        pytest.skip("GPU present")
    with pytest.raises(rt.RtError):
        rt.RtContext(dict(n=(2, 2, 2), x0=(0, 0, 0), dx=(1, 1, 1), bc_lo=("periodic",) * 3, bc_hi=("periodic",) * 3),
                     "minkowski", {}, 1)
