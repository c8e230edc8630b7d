"""The C-ABI library: loads, exports every symbol include/*.h declares, validates its arguments on the host
(no device needed for that) and fails loudly when there is no CUDA device (no CPU fallback)."""
import math
import os
import re
from dataclasses import replace

import pytest

from paper_1806_07938_b200 import tomo
from tomo_inputs.configs import WFS, get_config

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _declared():
    names = set()
    for h in ("tomo.h", "tomo_host.h"):
        src = open(os.path.join(ROOT, "include", h)).read()
        src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
        names |= set(re.findall(r"\b(tomo_[a-z0-9_]+)\s*\(", src))
    return names


def test_library_exports_every_declared_symbol():
    lib = tomo.load()
    declared = _declared()
    assert declared == set(tomo.EXPORTS), declared ^ set(tomo.EXPORTS)
    for name in declared:
        assert hasattr(lib, name), name


def _create(cfg, **kw):
    return tomo.TomoPlan(cfg, upload=False, **kw)


def test_argument_validation_happens_before_any_device_work():
    cfg = get_config("cfg1")
    with pytest.raises(tomo.TomoError) as e:
        _create(replace(cfg, frac=(0.7, 0.2)))
    assert e.value.code == tomo.TOMO_EINVAL and "sum to 1" in str(e.value)
    with pytest.raises(tomo.TomoError) as e:      # NGS + LGS in the high-order set: not 2RBT
        _create(replace(cfg, wfs=(WFS(10, 0), WFS(-10, 0, 90e3))))
    assert e.value.code == tomo.TOMO_EUNSUPPORTED
    with pytest.raises(tomo.TomoError) as e:      # two LGS altitudes
        _create(replace(cfg, wfs=(WFS(10, 0, 80e3), WFS(-10, 0, 90e3))))
    assert e.value.code == tomo.TOMO_EUNSUPPORTED
    with pytest.raises(tomo.TomoError) as e:      # layer above the guide star
        _create(replace(cfg, wfs=(WFS(10, 0, 4e3), WFS(-10, 0, 4e3))))
    assert e.value.code == tomo.TOMO_EINVAL
    with pytest.raises(tomo.TomoError) as e:      # pad below the linear-convolution support 2n-1
        _create(replace(cfg, pad=12))
    assert e.value.code == tomo.TOMO_EINVAL
    with pytest.raises(tomo.TomoError) as e:      # pad not 5-smooth
        _create(replace(cfg, pad=22))
    assert e.value.code == tomo.TOMO_EUNSUPPORTED
    with pytest.raises(tomo.TomoError) as e:
        _create(replace(cfg, wfs=(WFS(10, 0, math.inf, 1), WFS(-10, 0))))
    assert e.value.code == tomo.TOMO_EINVAL


def test_no_cpu_fallback():
    import torch
    if torch.cuda.is_available():
        pytest.skip("a CUDA device is present")
    with pytest.raises(tomo.TomoError) as e:
        _create(get_config("cfg1"))
    assert e.value.code == tomo.TOMO_ECUDA and "no CPU fallback" in str(e.value)
