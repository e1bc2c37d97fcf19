"""Tolerance rules for CUDA-vs-oracle parity (BASELINE.json north_star, readings 8c-13/14).

Plain rule, every plane P:   |d| <= max(1e-11 |P_ref|, 1e-13 max|P_ref|)
mu (ill-conditioned near critical lines):
    |d mu| <= 1e-11 |mu_ref| max(1, C),  C = ((1-kappa)^2 + gamma^2) |mu_ref|
    AND the plain rule on 1/mu.
"""
import numpy as np

REL, FLOOR = 1e-11, 1e-13


def conditioned_rel(ehat_max: float) -> float:
    """Relative tolerance for models whose largest e-hat is `ehat_max` (reading R20).

    The closed form itself loses digits as e-hat -> 1: the atanh argument tends to
    u = 2 sqrt(eps)/(1+eps) and d atanh/du = 1/(1-u^2) = ((1+eps)/(1-eps))^2 = 1/q^2 (q = axis
    ratio), so ONE rounding of u moves the result by 2^-53/q^2.  Against the 40-digit value the
    fp64 oracle itself is 4.7 x OUTSIDE the plain 1e-11 rule at e-hat = 0.9999 (q = 0.007) and
    at 0.40 of it at e-hat = 0.9992 (q = 0.02): pinned by
    tests/test_oracle_pins.py::test_r20_oracle_vs_40_digits_at_extreme_ellipticity.  The
    north-star 1e-11 holds for q >= 0.02 (e-hat <= 0.9992); beyond, 32 roundings of that size
    are allowed (the oracle uses 0.66 of that at e-hat = 0.9999)."""
    eps = ehat_max / (1.0 + np.sqrt(1.0 - ehat_max * ehat_max))
    q = (1.0 - eps) / (1.0 + eps)
    return max(REL, 32.0 * 2.0 ** -53 / (q * q))


def plain_violation(got, ref, rel=REL):
    """max over elements of |d| / allowed (<= 1 passes)."""
    got = np.asarray(got, dtype=np.float64)
    ref = np.asarray(ref, dtype=np.float64)
    if ref.size == 0:
        return 0.0
    allowed = np.maximum(rel * np.abs(ref), rel / REL * FLOOR * np.max(np.abs(ref)))
    allowed = np.maximum(allowed, 5e-324)
    d = np.abs(got - ref)
    d = np.where((got == ref), 0.0, d)  # equal infinities / zeros
    return float(np.max(d / allowed))


def mu_violation(mu_got, mu_ref, kappa_ref, g1_ref, g2_ref, rel=REL):
    mu_got = np.asarray(mu_got, dtype=np.float64)
    mu_ref = np.asarray(mu_ref, dtype=np.float64)
    C = ((1.0 - kappa_ref) ** 2 + g1_ref ** 2 + g2_ref ** 2) * np.abs(mu_ref)
    allowed = rel * np.abs(mu_ref) * np.maximum(1.0, C)
    fin = np.isfinite(mu_ref)
    v1 = float(np.max(np.abs(mu_got - mu_ref)[fin] / allowed[fin])) if fin.any() else 0.0
    assert np.array_equal(mu_got[~fin], mu_ref[~fin])
    with np.errstate(divide="ignore"):
        v2 = plain_violation(1.0 / mu_got, 1.0 / mu_ref, rel)
    return max(v1, v2)


def check_planes(got: dict, ref: dict, what="", rel=REL):
    """got/ref: name -> array. ref must hold kappa, gamma1, gamma2 when mu is compared."""
    worst = {}
    for n in got:
        if n == "mu":
            v = mu_violation(got["mu"], ref["mu"], ref["kappa"], ref["gamma1"], ref["gamma2"], rel)
        else:
            v = plain_violation(got[n], ref[n], rel)
        worst[n] = v
    bad = {n: v for n, v in worst.items() if not v <= 1.0}
    assert not bad, f"{what}: parity violated (|d|/allowed): {bad}"
    return worst


def stats_violation(mean_got, var_got, mean_ref, var_ref, nmodel: int):
    """Mean / variance of a plane over the models of a batch (lh_grid_stats_batch vs oracle.stats; R21).

    Each sample P_m is allowed the plain per-element error e = max(1e-11 |P_m|, 1e-13 max|plane|); per pixel
    |P_m| <= |mean| + sqrt(M var), so e <= max(1e-11 (|mean| + sqrt(M var)), 1e-13 max|mean plane|) =: E.
    mean: |d mean| <= E.   var = (1/M) sum (P_m - mean)^2: perturbing every sample by <= E moves it by at most
    2 sqrt(var) (2E) + (2E)^2 (Cauchy-Schwarz; the factor 2 covers the shift of the mean), plus the rounding of the
    sum itself, 1e-11 var.  Returns max |d| / allowed for (mean, var)."""
    mean_ref = np.asarray(mean_ref, dtype=np.float64)
    var_ref = np.asarray(var_ref, dtype=np.float64)
    fin = np.isfinite(mean_ref) & np.isfinite(var_ref)
    E = np.maximum(REL * (np.abs(mean_ref) + np.sqrt(nmodel * var_ref)), FLOOR * np.max(np.abs(mean_ref[fin])))
    am = np.maximum(E, 5e-324)
    av = 4.0 * np.sqrt(var_ref) * E + 4.0 * E * E + REL * var_ref
    vm = float(np.max(np.abs(mean_got - mean_ref)[fin] / am[fin]))
    vv = float(np.max(np.abs(var_got - var_ref)[fin] / np.maximum(av[fin], 5e-324)))
    return vm, vv


# ---------------------------------------------------------------- whole-map reports (tests/test_gpu_parity_full.py)
def plain_ratio_map(got, ref, rel=REL):
    """|d| / allowed of the plain rule, element by element (same rule as plain_violation)."""
    got = np.asarray(got, dtype=np.float64)
    ref = np.asarray(ref, dtype=np.float64)
    allowed = np.maximum(rel * np.abs(ref), rel / REL * FLOOR * np.max(np.abs(ref)))
    allowed = np.maximum(allowed, 5e-324)
    with np.errstate(invalid="ignore"):
        d = np.where(got == ref, 0.0, np.abs(got - ref))
    return d / allowed


def mu_ratio_map(mu_got, mu_ref, kappa_ref, g1_ref, g2_ref, rel=REL):
    """Element-wise max of the two ratios of the conditioned mu rule (reading R13); non-finite references must
    be reproduced exactly (ratio 0) or count as a violation (ratio inf)."""
    mu_got = np.asarray(mu_got, dtype=np.float64)
    mu_ref = np.asarray(mu_ref, dtype=np.float64)
    fin = np.isfinite(mu_ref)
    with np.errstate(invalid="ignore", divide="ignore", over="ignore"):
        C = ((1.0 - kappa_ref) ** 2 + g1_ref ** 2 + g2_ref ** 2) * np.abs(mu_ref)
        allowed = np.maximum(rel * np.abs(mu_ref) * np.maximum(1.0, C), 5e-324)
        r1 = np.where(fin, np.abs(mu_got - mu_ref) / allowed, np.where(mu_got == mu_ref, 0.0, np.inf))
        r2 = plain_ratio_map(1.0 / mu_got, 1.0 / mu_ref, rel)
    return np.maximum(r1, r2)


def mu_unconditioned_fraction(mu_got, mu_ref, rel=REL):
    """SURVEY sec. 8(c) pins table, last row: the fraction of pixels that ALSO pass the unconditioned test on mu.
    Returns (pure relative rule |d| <= rel |mu_ref|, plain rule with the 1e-13 max|mu| floor)."""
    mu_got = np.asarray(mu_got, dtype=np.float64)
    mu_ref = np.asarray(mu_ref, dtype=np.float64)
    with np.errstate(invalid="ignore"):
        d = np.where(mu_got == mu_ref, 0.0, np.abs(mu_got - mu_ref))
        pure = float(np.mean(d <= rel * np.abs(mu_ref)))
        fin = np.isfinite(mu_ref)
        floor = rel / REL * FLOOR * (np.max(np.abs(mu_ref[fin])) if fin.any() else 0.0)
        plain = float(np.mean(d <= np.maximum(rel * np.abs(mu_ref), floor)))
    return pure, plain


def report_planes(got: dict, ref: dict, rel=REL):
    """Whole-map report: name -> {worst, index (flat, of the worst element), n} and for mu the unconditioned
    pass fractions.  Nothing is asserted here; `worst <= 1` is the pass criterion of check_planes."""
    rep = {}
    for n in got:
        if n == "mu":
            r = mu_ratio_map(got["mu"], ref["mu"], ref["kappa"], ref["gamma1"], ref["gamma2"], rel)
        else:
            r = plain_ratio_map(got[n], ref[n], rel)
        r = np.where(np.isnan(r), np.inf, r)  # a NaN anywhere is a violation
        k = int(np.argmax(r))
        rep[n] = {"worst": float(r.reshape(-1)[k]), "index": k, "n": int(r.size)}
        if n == "mu":
            rep[n]["unconditioned_pure"], rep[n]["unconditioned_plain"] = mu_unconditioned_fraction(got["mu"], ref["mu"], rel)
    return rep
