"""Accuracy of the kernels' own fp64 routines (csrc/ep_math.cuh) on the device, against mpmath / numpy references.

The claims in ep_math.cuh: 2^x relative error <= 4.2e-16, <= 3.1 ulp (degree-9 minimax polynomial, 3e-16), log <= 1 ulp where |log x| > 1 (the concentrations) and <= 2.5 ulp near x = 1,
rcp <= 1 ulp, rsqrt <= 2 ulp.
"""
import numpy as np
import pytest

from ep_inputs.prng import uniform

pytestmark = pytest.mark.gpu


def _ulp_err(got, ref_hi):
    """|got - ref| in units of the last place of ref; ref_hi is a longdouble (64-bit mantissa) reference."""
    ref = ref_hi.astype(np.float64)
    return np.abs((got.astype(np.longdouble) - ref_hi) / np.spacing(np.abs(ref)).astype(np.longdouble)).astype(np.float64)


def test_exp2_accuracy():
    """The kernels' exponential primitive is 2^x (log2(e) is folded into the compile-time slopes of every exponent)."""
    import paper_2112_12854_b200 as ep
    n = 400000
    x = np.concatenate([uniform(1, np.arange(n), -1000.0, 1000.0), uniform(2, np.arange(n), -60.0, 60.0),
                        uniform(3, np.arange(n), -1.0, 1.0), uniform(4, np.arange(n), -1e-3, 1e-3),
                        np.array([0.0, -0.0, 1000.0, -1000.0, 0.5, -0.5, 1e-300, 0.49999999999999994, 1.0, -1.0, 10.0])])
    y = ep.math_eval(0, x)
    err = _ulp_err(y, np.exp2(x.astype(np.longdouble)))
    assert err.max() <= 3.2, err.max()
    rel = np.abs((y.astype(np.longdouble) - np.exp2(x.astype(np.longdouble))) / np.exp2(x.astype(np.longdouble))).astype(np.float64)
    assert rel.max() <= 4.2e-16, rel.max()
    assert y[x == 0.0].tolist() == [1.0, 1.0]
    assert ep.math_eval(0, np.array([1.0, -1.0, 10.0])).tolist() == [2.0, 0.5, 1024.0]    # integer arguments are exact
    assert np.all(np.diff(ep.math_eval(0, np.linspace(-5, 5, 200001))) >= 0)      # monotone on a fine grid


def test_log_accuracy():
    import paper_2112_12854_b200 as ep
    n = 400000
    x = np.concatenate([uniform(5, np.arange(n), 1e-6, 1e-2), uniform(6, np.arange(n), 3.0, 30.0),
                        uniform(7, np.arange(n), 100.0, 200.0), uniform(8, np.arange(n), 0.5, 2.0),
                        np.array([1.0, 2.0, 0.5, np.sqrt(2.0), np.nextafter(np.sqrt(2.0), 2.0), 1e-300, 1e300])])
    y = ep.math_eval(1, x)
    ref = np.log(x.astype(np.longdouble))
    absref = np.abs(ref.astype(np.float64))
    err = _ulp_err(y, ref)
    assert err[absref > 1e-3].max() <= 2.5, err[absref > 1e-3].max()     # s = (m-1)/(m+1) carries two roundings
    assert err[: 3 * n].max() <= 1.0, err[: 3 * n].max()                  # the ranges of Ca_i, Na_i, K_i: |log x| > 1
    assert np.abs(y - ref.astype(np.float64))[absref <= 1e-3].max() <= 3e-19     # near x = 1: absolute accuracy
    assert y[x == 1.0][0] == 0.0


def test_rcp_and_rsqrt_accuracy():
    import paper_2112_12854_b200 as ep
    n = 400000
    x = np.concatenate([uniform(9, np.arange(n), 1e-8, 1.0), uniform(10, np.arange(n), 1.0, 1e12),
                        -uniform(11, np.arange(n), 1e-3, 1e3), np.array([1.0, 2.0, 3.0, 1e-200, 1e200])])
    r = ep.math_eval(2, x)
    assert _ulp_err(r, 1.0 / x.astype(np.longdouble)).max() <= 1.0
    xp = x[x > 0]
    q = ep.math_eval(3, xp)
    assert _ulp_err(q, 1.0 / np.sqrt(xp.astype(np.longdouble))).max() <= 2.0
