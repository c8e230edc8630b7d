"""tomo_apply_css_static (include/tomo.h): the covariance product with its whole workspace in the library's file-scope device
array -- for callers that may not allocate -- against the existing path tomo_apply_css on the same plan and input.

Collected last on purpose (the suite runs with pytest -x).  Passes alone in a fresh process and after the other GPU tests:
every call clears the part of the shared array it uses, so neither order nor an earlier plan's data matters.

Gates: the multi-kernel solver runs the same kernels in the same order -> bitwise equal; against the persistent kernel's
single-product launch the product gate of tests/gates.py (rel-L2 <= 1e-4, max-abs <= 1e-5 rms, P-a)."""
from dataclasses import replace

import numpy as np
import pytest

torch = pytest.importorskip("torch")

from paper_1806_07938_b200 import tomo  # noqa: E402
from tomo_inputs.configs import get_config, small_lgs_config  # noqa: E402

from gates import assert_close  # noqa: E402

pytestmark = pytest.mark.gpu


def _vec(plan, seed):
    g = torch.Generator(device="cpu").manual_seed(seed)
    return torch.randn(plan.slopes_len, generator=g, dtype=torch.float32).cuda()


def _both(plan, v):
    want = torch.empty(plan.slopes_len, dtype=torch.float32, device="cuda")
    got = torch.full((plan.slopes_len,), float("nan"), dtype=torch.float32, device="cuda")
    plan.apply_css(v, want)
    plan.apply_css_static(v, got)
    torch.cuda.synchronize()
    return got.cpu().numpy(), want.cpu().numpy()


@pytest.mark.parametrize("name", ["small_lgs_focus", "cfg2", "cfg3"])
def test_static_scratch_product_equals_the_existing_path_on_two_calls_in_a_row(name):
    cfg = (replace(small_lgs_config(n=11, n_gs=3, n_layers=2, n_remove=3), obstruction=0.3) if name == "small_lgs_focus"
           else get_config(name))
    p_mk = tomo.TomoPlan(cfg, build_cos=False, solver=tomo.TOMO_SOLVER_MULTIKERNEL)
    p_ps = tomo.TomoPlan(cfg, build_cos=False, solver=tomo.TOMO_SOLVER_PERSISTENT)
    assert p_mk.solver_in_use()[0] == tomo.TOMO_SOLVER_MULTIKERNEL and p_ps.solver_in_use()[0] == tomo.TOMO_SOLVER_PERSISTENT
    before = p_mk.stats()["device_bytes"]
    for call, seed in enumerate((1, 2)):                        # two calls in a row, different inputs: the second runs on the
        v = _vec(p_mk, seed)                                    # array as the first left it
        got, want = _both(p_mk, v)
        assert np.isfinite(got).all() and np.array_equal(got, want), (name, "multi-kernel", call)
        got, want = _both(p_ps, v)
        assert_close(got, want, 1e-4, what=(name, "persistent", call))
    # the same input again after another plan used the array: bitwise the first answer
    v = _vec(p_mk, 1)
    first, _ = _both(p_mk, v)
    _both(p_ps, _vec(p_ps, 3))
    again, _ = _both(p_mk, v)
    assert np.array_equal(first, again)
    assert p_mk.stats()["device_bytes"] == before               # the plan allocated nothing for it
    p_mk.close()
    p_ps.close()


def test_static_scratch_product_in_the_other_precisions():
    cfg = get_config("cfg2")
    for prec in (tomo.TOMO_F32S_F64A, tomo.TOMO_F64):
        pl = tomo.TomoPlan(cfg, build_cos=False, solver=tomo.TOMO_SOLVER_MULTIKERNEL, precision=prec)
        for seed in (4, 5):
            got, want = _both(pl, _vec(pl, seed))
            assert np.array_equal(got, want), prec
        pl.close()


def test_a_plan_larger_than_the_static_scratch_is_refused_with_both_sizes_named():
    cfg = get_config("cfg4")                                    # C = 16, n = 74, fp64: 4.2 MB of workspace > 4 MiB
    pl = tomo.TomoPlan(cfg, build_cos=False, precision=tomo.TOMO_F64)
    v = _vec(pl, 6)
    out = torch.zeros(pl.slopes_len, dtype=torch.float32, device="cuda")
    with pytest.raises(tomo.TomoError) as e:
        pl.apply_css_static(v, out)
    torch.cuda.synchronize()
    assert e.value.code == tomo.TOMO_EINVAL and str(tomo.TOMO_STATIC_SCRATCH_BYTES) in str(e.value) and "tomo_apply_css" in str(e.value)
    assert float(out.abs().max()) == 0.0                        # nothing was launched
    pl.close()
    p32 = tomo.TomoPlan(cfg, build_cos=False)                   # the same system in fp32 fits (2.1 MB)
    got, want = _both(p32, _vec(p32, 7))
    assert_close(got, want, 1e-4, what="cfg4 fp32")
    p32.close()
