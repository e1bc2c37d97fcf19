"""NEXT row f3 on the GPU: lh_chi2 vs oracle.chi2 (-m gpu), through the C ABI.

The constraints of the cluster case are made with the ORACLE (true model -> random sources -> oracle.delens ->
images with at least two per source, plus seeded noise): no input comes from the CUDA path.  The two sides compute
their own deflections (1e-13 apart), so chi^2 and the predicted positions are compared to 1e-8 relative /
1e-9 arcsec; the no-lens cases are exact."""
import numpy as np
import pytest

import lens_inputs as li
import oracle
import paper_2004_06352_b200 as lh

pytestmark = pytest.mark.gpu
torch = pytest.importorskip("torch")


def gpu_chi2(L, g, c, nsrc):
    chi = torch.full((1,), float("nan"), dtype=torch.float64, device="cuda")
    pred = torch.full((max(len(c), 1), 2), 7.0, dtype=torch.float64, device="cuda")
    src = torch.full((max(nsrc, 1), 2), 7.0, dtype=torch.float64, device="cuda")
    nim = torch.full((1,), -1, dtype=torch.int64, device="cuda")
    lh.lh_chi2(L, g, c, nsrc, chi, pred, src, nim)
    torch.cuda.synchronize()
    return {"chi2": float(chi.item()), "predicted": pred.cpu().numpy()[: len(c)], "sources": src.cpu().numpy()[:nsrc],
            "nimages": int(nim.item())}


def test_no_lens_cases_are_exact():
    g = li.Grid(x0=-4.0, y0=-4.0, dx=0.5, nx=17, ny=17)
    none = li.make_lenses(0)
    c = li.make_constraints([(0, 1.1, 0.3, 0.5), (0, -0.7, 1.9, 0.25), (1, 2.2, -2.3, 1.0), (3, 0.4, 0.4, 2.0)])
    got, want = gpu_chi2(none, g, c, 4), oracle.chi2(none, g.x0, g.y0, g.dx, g.nx, g.ny, c, 4)
    assert got["chi2"] == want["chi2"] and got["nimages"] == want["nimages"] == 3
    assert np.array_equal(got["predicted"], want["predicted"])
    assert np.array_equal(got["sources"], want["sources"], equal_nan=True) and np.isnan(got["sources"][2]).all()
    far = li.make_constraints([(0, 50.0, 50.0, 0.1)])  # no predicted image on the grid -> +inf
    assert gpu_chi2(none, g, far, 1)["chi2"] == np.inf
    assert gpu_chi2(none, g, li.make_constraints([]), 0)["chi2"] == 0.0  # nothing to fit


def _cluster_constraints(c, g, nsrc, seed):
    rng = np.random.default_rng(seed)
    ref = oracle.grid(c.lenses, g.x0, g.y0, g.dx, g.nx, g.ny, planes=("ax", "ay"), threads=8)
    half = 0.25 * g.nx * g.dx / 2
    src = np.column_stack([rng.uniform(-half, half, nsrc), rng.uniform(-half, half, nsrc)])
    im, _ = oracle.delens(ref["ax"], ref["ay"], g.x0, g.y0, g.dx, src)
    rows, ns = [], 0
    for s in range(nsrc):
        mine = im[im["source"] == s]
        if len(mine) < 2:
            continue
        for r in mine:
            rows.append((ns, r["x"] + 0.05 * rng.standard_normal(), r["y"] + 0.05 * rng.standard_normal(), 0.3))
        ns += 1
    return li.make_constraints(rows), ns


@pytest.mark.parametrize("perturb", [False, True])
def test_cluster_chi2_matches_oracle(perturb):
    c = li.config(1, scale=4)  # 256 x 256, 100 dPIE
    g = c.grid
    cons, ns = _cluster_constraints(c, g, 40, seed=5)
    assert ns >= 5 and len(cons) >= 2 * ns
    L = c.lenses.copy()
    if perturb:  # the model under test is off: halo 0 heavier and shifted
        L["b0"][0] *= 1.05
        L["x"][0] += 0.5
    got = gpu_chi2(L, g, cons, ns)
    want = oracle.chi2(L, g.x0, g.y0, g.dx, g.nx, g.ny, cons, ns)
    assert np.isfinite(want["chi2"]) and want["chi2"] > 0
    assert abs(got["chi2"] - want["chi2"]) <= 1e-8 * want["chi2"]
    assert np.allclose(got["sources"], want["sources"], rtol=0, atol=1e-10)
    assert np.allclose(got["predicted"], want["predicted"], rtol=0, atol=1e-9)
    assert abs(got["nimages"] - want["nimages"]) <= 2


def test_chi2_argument_errors():
    g = li.Grid(x0=-4.0, y0=-4.0, dx=0.5, nx=17, ny=17)
    chi = torch.full((1,), float("nan"), dtype=torch.float64, device="cuda")
    for bad in ([(2, 0.0, 0.0, 1.0)], [(0, 0.0, 0.0, 0.0)], [(0, float("nan"), 0.0, 1.0)], [(-1, 0.0, 0.0, 1.0)]):
        with pytest.raises(lh.LhError):
            lh.lh_chi2(li.make_lenses(0), g, li.make_constraints(bad), 2, chi)
    badlens = li.lens(li.DPIE, 0, 0, 0.3, 0.1, 0.1, 0.05, 1.0)  # rcut < rcore
    with pytest.raises(lh.LhError):
        lh.lh_chi2(badlens, g, li.make_constraints([(0, 0.0, 0.0, 1.0)]), 1, chi)
    torch.cuda.synchronize()
    assert torch.isnan(chi).all()


def test_chi2_on_two_streams_does_not_share_scratch_unsafely():
    """lh_chi2 keeps its scratch (deflection planes, sources, image list, counter) in ONE cached buffer per device.
    Calls on different streams must not overwrite it while an earlier call is still running: the second stream waits
    for the first call's end event.  Two different problems alternate on two streams, several times, each result is
    compared with the result of the same call made alone."""
    c = li.config(1, scale=4)
    g = c.grid
    cons_a, ns_a = _cluster_constraints(c, g, 40, seed=5)
    cons_b, ns_b = _cluster_constraints(c, g, 30, seed=9)
    Lb = c.lenses.copy()
    Lb["b0"][0] *= 1.05
    alone_a, alone_b = gpu_chi2(c.lenses, g, cons_a, ns_a), gpu_chi2(Lb, g, cons_b, ns_b)
    s1, s2 = torch.cuda.Stream(), torch.cuda.Stream()
    outs = []
    torch.cuda.synchronize()
    try:
        for k in range(4):
            for st, (L, cons, ns) in ((s1, (c.lenses, cons_a, ns_a)), (s2, (Lb, cons_b, ns_b))):
                chi = torch.full((1,), float("nan"), dtype=torch.float64, device="cuda")
                pred = torch.full((len(cons), 2), 7.0, dtype=torch.float64, device="cuda")
                nim = torch.full((1,), -1, dtype=torch.int64, device="cuda")
                lh.lh_set_stream(st)
                lh.lh_chi2(L, g, cons, ns, chi, pred, None, nim)
                outs.append((chi, pred, nim))
    finally:
        lh.lh_set_stream(None)
    torch.cuda.synchronize()
    for k, (chi, pred, nim) in enumerate(outs):
        want = alone_a if k % 2 == 0 else alone_b
        assert float(chi.item()) == want["chi2"] and int(nim.item()) == want["nimages"]
        assert np.array_equal(pred.cpu().numpy(), want["predicted"])
