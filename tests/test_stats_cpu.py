"""Pins of oracle.stats (mean / population variance of maps over the models of a batch; R21)
against closed forms -- CPU only."""
import numpy as np

import lens_inputs as li
import oracle

G = li.Grid(x0=-7.0, y0=-5.0, dx=1.0, nx=15, ny=11)
PL = ("ax", "kappa", "gamma1")


def _maps(L):
    return oracle.grid(L, G.x0, G.y0, G.dx, G.nx, G.ny, planes=PL)


def test_single_model_mean_is_the_map_and_variance_zero():
    L = li.config(0).lenses
    mean, var = oracle.stats(L, 1, len(L), G.x0, G.y0, G.dx, G.nx, G.ny, planes=PL)
    ref = _maps(L)
    for n in PL:
        assert np.array_equal(mean[n], ref[n]) and np.all(var[n] == 0.0)


def test_two_models_closed_form():
    """M = 2: mean = (a+b)/2, var = ((a-b)/2)^2."""
    A, B = li.config(0).lenses, li.cluster(9, 0, 10, 40.0)
    mean, var = oracle.stats(np.concatenate([A, B]), 2, 10, G.x0, G.y0, G.dx, G.nx, G.ny, planes=PL)
    a, b = _maps(A), _maps(B)
    for n in PL:
        assert np.allclose(mean[n], 0.5 * (a[n] + b[n]), rtol=1e-15, atol=0)
        assert np.allclose(var[n], (0.5 * (a[n] - b[n])) ** 2, rtol=1e-12, atol=1e-30)


def test_b0_scaling_family_closed_form():
    """Models that differ only by an overall factor s_m on every b0: every plane is linear in b0 (alpha, Hessian,
    kappa, gamma), so P_m = s_m P_1 and mean = mean(s) P_1, var = var(s) P_1^2."""
    base = li.config(0).lenses
    s = np.array([1.0, 0.5, 2.0, 1.25, 0.75])
    Ls = []
    for f in s:
        L = base.copy()
        L["b0"] *= f
        Ls.append(L)
    mean, var = oracle.stats(np.concatenate(Ls), len(s), len(base), G.x0, G.y0, G.dx, G.nx, G.ny, planes=PL)
    p1 = _maps(base)
    ms, vs = s.mean(), ((s - s.mean()) ** 2).mean()
    for n in PL:
        assert np.allclose(mean[n], ms * p1[n], rtol=1e-14, atol=0)
        assert np.allclose(var[n], vs * p1[n] ** 2, rtol=1e-12, atol=0)


def test_order_of_models_does_not_matter_and_repeats_give_zero_variance():
    A, B, Cc = li.config(0).lenses, li.cluster(9, 0, 10, 40.0), li.cluster(10, 0, 10, 40.0)
    m1, v1 = oracle.stats(np.concatenate([A, B, Cc]), 3, 10, G.x0, G.y0, G.dx, G.nx, G.ny, planes=PL)
    m2, v2 = oracle.stats(np.concatenate([Cc, A, B]), 3, 10, G.x0, G.y0, G.dx, G.nx, G.ny, planes=PL)
    for n in PL:
        assert np.allclose(m1[n], m2[n], rtol=1e-14) and np.allclose(v1[n], v2[n], rtol=1e-11, atol=1e-30)
    m3, v3 = oracle.stats(np.concatenate([A, A, A, A]), 4, 10, G.x0, G.y0, G.dx, G.nx, G.ny, planes=PL)
    for n in PL:
        assert np.array_equal(m3[n], _maps(A)[n]) and np.all(v3[n] == 0.0)
