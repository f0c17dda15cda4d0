"""P7: the oracle's geometric source terms (O6) against the covariant expressions of the paper.

PAPER.md:54 (eq. 2): the momentum source is sqrt(-g) T^kappa_lambda Gamma^lambda_{j kappa}.  Here that
expression is evaluated in four dimensions (numpy, Christoffel symbols from exact complex-step derivatives of
the closed-form Kerr-Schild metric) and compared with the oracle's 3+1 formula.  The energy source of the
tau equation is pinned to the projection n_nu nabla_mu T^{mu nu} = 0 written out covariantly:
alpha sqrt(gamma) (T^{i0} d_i alpha - alpha T^{mu nu} Gamma^0_{mu nu}) for a stationary metric.
"""
import numpy as np

import workloads as wl
from oracle import binding as ob
from helpers4d import SYM, christoffel, fluid4, gamma3, metric4

GAM = 4.0 / 3.0


def ks_met10(x):
    a, b, g = wl.kerr_schild(x[0], x[1], x[2])
    return np.array([a, b[0], b[1], b[2], *g])


def ks_dmet(x):
    """Exact derivatives d_j met10 by the complex-step method (the closed form is analytic)."""
    out = np.zeros((3, 10))
    for j in range(3):
        xc = np.array(x, dtype=complex)
        xc[j] += 1e-30j
        out[j] = np.imag(ks_met10(xc)) / 1e-30
    return out


def metric4_derivs(m, dm):
    """d_k g_{mu nu} (k = 0..3; k = 0 vanishes: stationary) from derivatives of alpha, beta^i, gamma_ij."""
    dG = np.zeros((4, 4, 4))
    al, be, g = m[0], m[1:4], gamma3(m)
    for j in range(3):
        dal, dbe, dg = dm[j][0], dm[j][1:4], gamma3(dm[j])
        dbl = dg @ be + g @ dbe
        dG[1 + j, 0, 0] = -2 * al * dal + dbe @ (g @ be) + be @ dbl
        dG[1 + j, 0, 1:] = dG[1 + j, 1:, 0] = dbl
        dG[1 + j, 1:, 1:] = dg
    return dG


def test_sources_equal_covariant_expressions_on_kerr_schild():
    rng = np.random.default_rng(7)
    P, _ = wl.random_states(71, 200)
    worst = 0.0
    for q in P:
        x = rng.uniform(-8, 8, 3)
        while np.linalg.norm(x) < 3.0:
            x = rng.uniform(-8, 8, 3)
        m = ks_met10(x)
        dm = ks_dmet(x)
        # keep the state physical in this metric: rescale ut to |v| < 0.95
        g = gamma3(m)
        q = q.copy()
        f = fluid4(q, m, GAM)
        G, T = f["G"], f["T"]
        dG = metric4_derivs(m, dm)
        # check the assembled derivative against a direct complex step of the 4-metric
        for j in range(3):
            xc = np.array(x, dtype=complex); xc[j] += 1e-30j
            assert np.allclose(np.imag(metric4(ks_met10(xc))) / 1e-30, dG[1 + j], rtol=1e-12, atol=1e-14)
        Gam4 = christoffel(G, dG)
        Tmix = T @ G                                    # T^kappa_lambda
        sqrtmg = m[0] * np.sqrt(np.linalg.det(g))
        srcS = np.array([sqrtmg * np.einsum("kl,lk->", Tmix, Gam4[:, 1 + j, :]) for j in range(3)])
        srcTau = sqrtmg * (T[1:, 0] @ dm[:, 0] - m[0] * np.einsum("mn,mn->", T, Gam4[0]))
        got = ob.source_point(q, m, dm.ravel(), GAM)
        sc = sqrtmg * np.abs(T).max() * np.abs(dG).max()
        worst = max(worst, np.abs(got[:3] - srcS).max() / sc, abs(got[3] - srcTau) / sc)
    assert worst < 1e-12, worst


def test_sources_vanish_identically_in_flat_space():
    """P5: alpha = 1, beta = 0, gamma = delta, zero derivatives: every source is exactly 0.0."""
    P, _ = wl.random_states(72, 50)
    flat = np.array([1, 0, 0, 0, 1, 0, 0, 1, 0, 1.0])
    for q in P:
        assert np.all(ob.source_point(q, flat, np.zeros(30), GAM) == 0.0)


def test_kerr_schild_closed_form():
    """P10: alpha sqrt(gamma) = 1, gamma^{ij} = delta - 2H l l/(1+2H), beta^i = 2H l^i/(1+2H), l.l = 1."""
    rng = np.random.default_rng(3)
    for _ in range(200):
        x = rng.uniform(-10, 10, 3)
        if np.linalg.norm(x) < 2.5:
            continue
        m = ks_met10(x)
        g = gamma3(m)
        assert np.isclose(m[0] * np.sqrt(np.linalg.det(g)), 1.0, rtol=1e-13)
        twoH = 1 / m[0] ** 2 - 1
        l = m[1:4] * (1 + twoH) / twoH
        assert np.isclose(l @ l, 1.0, rtol=1e-12)
        assert np.allclose(np.linalg.inv(g), np.eye(3) - twoH * np.outer(l, l) / (1 + twoH), atol=1e-12)
        # the 4-metric is eta + 2H l l with l null: inverse is eta - 2H l l
        G = metric4(m)
        l4 = np.array([1, *l])
        assert np.allclose(G, np.diag([-1, 1, 1, 1.0]) + twoH * np.outer(l4, l4), atol=1e-12)
