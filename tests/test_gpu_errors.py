"""Error behaviour of the C ABI on the GPU box (include/dwf.h: status codes, no abort, message in dwf_last_error)."""
import ctypes

import numpy as np
import pytest

from paper_2203_17119_b200 import inputs

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def ctx():
    import torch
    assert torch.cuda.is_available()
    from paper_2203_17119_b200 import api
    g = api.Dwf((4, 4, 4, 8), 8, 1.8, 0.01, 1.5, 0.5)
    yield api, g
    g.close()


def test_operators_need_a_gauge_field(ctx):
    api, g = ctx
    a, b = g.new_native(api.F64, api.ODD), g.new_native(api.F64, api.EVEN)
    with pytest.raises(api.DwfError) as e:
        g.dhop(a, api.EVEN, False, api.F64, out=b)
    assert e.value.status == api.ESTATE and "gauge" in str(e.value)
    with pytest.raises(api.DwfError) as e:
        g.cg(a, 1e-8, 10)
    assert e.value.status == api.ESTATE


def test_aliasing_bad_tolerance_and_late_options(ctx):
    api, g = ctx
    g.set_gauge(inputs.gauge_weak((4, 4, 4, 8), 0.3, 5))
    a = g.new_native(api.F64, api.ODD).normal_()
    for call in (lambda: g.mpc(a, False, api.F64, out=a), lambda: g.mdagm(a, api.F64, out=a),
                 lambda: g.mooee_inv(a, api.ODD, False, api.F64, out=a)):
        with pytest.raises(api.DwfError) as e:
            call()
        assert e.value.status == api.EINVAL
    info = api.CgInfo()
    st = g.lib.dwf_cg(g._h, g._p(g.new_native()), g._p(a), -1.0, 10, api.CG_F64, 0, ctypes.byref(info))
    assert st == api.EINVAL
    full = g.new_native(api.F64, api.FULL).normal_()
    for fn in (lambda: g.lib.dwf_cg(g._h, g._p(g.new_native()), g._p(a), 1e-8, -1, api.CG_F64, 0, ctypes.byref(info)),
               lambda: g.lib.dwf_solve(g._h, g._p(g.new_native(api.F64, api.FULL)), g._p(full), 1e-8, -1, api.CG_F64,
                                       ctypes.byref(info))):
        assert fn() == api.EINVAL                      # a negative iteration budget is a bad argument everywhere
    with pytest.raises(api.DwfError) as e:
        g.set_option("compress12", 0)                  # layout options are frozen once the gauge field is in
    assert e.value.status == api.ESTATE
    with pytest.raises(api.DwfError) as e:
        g.set_option("no_such_option", 1)
    assert e.value.status == api.EINVAL


def test_max_iter_reached_is_reported_not_raised(ctx):
    api, g = ctx
    b = g.pack(inputs.source_half((4, 4, 4, 8), 8, 9, parity=1), api.F64, api.ODD)
    x, info, st = g.cg(b, 1e-12, 3, api.CG_F64)
    assert st == api.ENOTCONV and info["iters_total"] == 3 and info["resid_true"] > 1e-12
    assert np.isfinite(g.unpack(x, api.F64, api.ODD)).all()        # x holds the best iterate
    x, info, st = g.cg(g.new_native().zero_(), 1e-10, 100, api.CG_F64)      # b = 0: x = 0, converged at once
    assert st == api.OK and info["iters_total"] == 0 and float(x.abs().max()) == 0.0


def test_two_row_links_must_be_su3_and_probe_knobs_are_not_in_the_product(oracle_built):
    """2-row compression (reading C10) rebuilds row 2 as conj(row0 x row1), which is only right for SU(3):
    anything else is refused at dwf_set_gauge instead of silently giving another operator; 18-real storage takes it."""
    import torch
    from paper_2203_17119_b200 import api
    from oracle.dwf_oracle import Oracle
    dims, Ls = (4, 4, 4, 4), 4
    U = inputs.gauge_weak(dims, 0.3, 5)
    bad = U.copy()
    bad[1, 2, 3, 0, 2] *= 1.5                      # one link scaled: unitary up to a factor, not SU(3)
    g = api.Dwf(dims, Ls, 1.8, 0.1, 1.5, 0.5)
    with pytest.raises(api.DwfError) as e:
        g.set_gauge(bad)
    assert e.value.status == api.EINVAL and "SU(3)" in str(e.value)
    g.set_gauge(U)                                  # the context is still usable
    g.close()
    g = api.Dwf(dims, Ls, 1.8, 0.1, 1.5, 0.5, compress12=0)
    g.set_gauge(bad)
    src = inputs.source_half(dims, Ls, 3, parity=1)
    got = g.unpack(g.dhop(g.pack(src, api.F64, api.ODD), api.EVEN, False, api.F64), api.F64, api.EVEN)
    want = Oracle(dims, Ls, 1.8, 0.1, 1.5, 0.5).set_gauge(bad).dhop(src, 0, False)
    assert np.linalg.norm((got - want).ravel()) / np.linalg.norm(want.ravel()) < 1e-12
    # the measurement knobs of the probe build are not options of the product library
    for key in ("dhop_skip", "dhop_grid", "dhop_order", "dhop_sc"):
        with pytest.raises(api.DwfError) as e:
            g.set_option(key, 1)
        assert e.value.status == api.EINVAL
    g.close()
