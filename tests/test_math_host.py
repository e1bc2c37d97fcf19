"""The kernel's own FP64 primitives (csrc/lh_math.cuh), evaluated on the HOST through
lh_math_host_eval and pinned against mpmath / numpy -- no GPU, no oracle involved.
DESIGN.md sec. 6: seed + one third-order step is good to a few ulp; atan / atanh reduce
against a table and keep |z| <= 2^-8."""
import numpy as np
import pytest

import paper_2004_06352_b200 as lh

mp = pytest.importorskip("mpmath")
mp.mp.dps = 40
ULP = 2.0 ** -52


def rel_err(got, want):
    want = np.asarray(want, dtype=np.float64)
    return np.max(np.abs(got - want) / np.maximum(np.abs(want), 1e-300))


def test_rcp_sqrt_rsqrt_few_ulp():
    rng = np.random.default_rng(0)
    x = np.exp(rng.uniform(-60, 60, 20000))
    assert rel_err(lh.lh_math_host_eval(0, x), 1.0 / x) < 2 * ULP
    assert rel_err(lh.lh_math_host_eval(1, x), np.sqrt(x)) < 2 * ULP
    assert rel_err(lh.lh_math_host_eval(2, x), 1.0 / np.sqrt(x)) < 2 * ULP
    xn = -x
    assert rel_err(lh.lh_math_host_eval(0, xn), 1.0 / xn) < 2 * ULP


def test_shared_seed_reciprocals():
    rng = np.random.default_rng(1)
    a = np.exp(rng.uniform(-20, 20, 20000))
    b = np.exp(rng.uniform(-20, 20, 20000))
    assert rel_err(lh.lh_math_host_eval(5, a, b), 1.0 / a) < 4 * ULP
    assert rel_err(lh.lh_math_host_eval(6, a, b), 1.0 / a) < 6 * ULP


def _mp_vec(f, n, d):
    return np.array([float(f(mp.mpf(float(a)) / mp.mpf(float(b)))) for a, b in zip(n, d)])


def test_atan_whole_range():
    rng = np.random.default_rng(2)
    # quotients from 1e-300 to 1e+12, both signs, plus exact table nodes and octave edges
    q = np.concatenate([np.exp(rng.uniform(-30, 30, 4000)), 2.0 ** np.arange(-12, 13), [0.0, 1e-300, 1e12, 253.9, 256.0, 300.0],
                        2.0 ** -8 * (1 + np.arange(64) / 64.0)])
    d = np.exp(rng.uniform(-10, 10, q.size))
    n = q * d * np.where(rng.random(q.size) < 0.5, -1.0, 1.0)
    got = lh.lh_math_host_eval(3, n, d)
    want = _mp_vec(mp.atan, n, d)
    assert rel_err(got, want) < 4 * ULP
    assert np.all(np.signbit(got) == np.signbit(n))
    # tiny stand-in numerator of the circular limit (lh_pack.cpp): atan(u) = u exactly
    tiny = lh.lh_math_host_eval(3, np.array([2.0 ** -500 * 3.0]), np.array([7.0]))
    assert tiny[0] == 2.0 ** -500 * 3.0 / 7.0


def test_atanh_whole_table_range():
    rng = np.random.default_rng(3)
    # u = n/d with (1+u)/(1-u) from 1 to just below 2^16
    ratio = np.concatenate([np.exp(rng.uniform(0, np.log(65000.0), 4000)), [1.0, 1.0 + 1e-15, 2.0, 65535.0],
                            1.0 + np.arange(64) / 64.0])
    u = (ratio - 1.0) / (ratio + 1.0)
    d = np.exp(rng.uniform(-10, 10, u.size))
    n = u * d * np.where(rng.random(u.size) < 0.5, -1.0, 1.0)
    got = lh.lh_math_host_eval(4, n, d)
    want = _mp_vec(mp.atanh, n, d)
    # conditioning of atanh in its argument grows like 1/(1-u^2); the primitive itself stays within a few ulp of
    # the value at the (rounded) inputs it was given
    assert rel_err(got, want) < 6 * ULP
    assert np.all(np.signbit(got) == np.signbit(n))
    assert lh.lh_math_host_eval(4, np.array([0.0]), np.array([3.0]))[0] == 0.0


def test_bad_arguments():
    with pytest.raises(lh.LhError):
        lh.lh_math_host_eval(9, np.ones(3))
    with pytest.raises(lh.LhError):
        lh.lh_math_host_eval(3, np.ones(3))  # atan needs both arrays
