"""Pins of the oracle's per-state formulas (O1-O5, O8) against things the paper and mathematics fix.

The paper prints only the covariant system (eqs. 1-2); every pin here compares the
oracle's 3+1 formulas with an INDEPENDENT evaluation from those covariant definitions (tests/helpers4d.py),
with brute force, or with closed-form limits.  None of them re-types the oracle's own expression.
"""
import numpy as np
import pytest

import workloads as wl
from oracle import OracleParams
from oracle import binding as ob
from helpers4d import fluid4, gamma3, metric4

GAM = 4.0 / 3.0


def states(seed, n, **kw):
    return wl.random_states(seed, n, **kw)


# ---- O1: conserved variables are sqrt(-g) J^t and sqrt(-g) T^t_mu ---------------
def test_prim2con_matches_covariant_definitions():
    P, M = states(11, 300)
    for q, m in zip(P, M):
        f = fluid4(q, m, GAM)
        al = m[0]
        be = m[1:4]
        T, G = f["T"], f["G"]
        w = ob.prim2con_point(q, m, GAM)
        D = al * q[0] * f["u"][0]                       # sqrt(-g) J^t / sqrt(gamma)
        Tt_low = T[0] @ G                                # T^t_mu
        S = al * Tt_low[1:]                              # alpha T^t_j
        tau = al * al * T[0, 0] - D                      # n_mu n_nu T^{mu nu} - D
        # the paper's energy variable: -sqrt(-g) T^t_t = alpha (tau + D) - beta^j S_j   (per sqrt(gamma))
        assert np.isclose(-al * Tt_low[0], al * (w[4] + w[0]) - be @ w[1:4], rtol=1e-12, atol=1e-300)
        scale = abs(tau) + abs(D)
        assert abs(w[0] - D) <= 1e-13 * abs(D)
        assert np.allclose(w[1:4], S, rtol=0, atol=1e-12 * (np.abs(S).max() + scale))
        assert abs(w[4] - tau) <= 1e-12 * scale
        # B^i = alpha *F^{it}
        assert np.allclose(w[5:8], al * f["Fdual"][1:, 0], rtol=0, atol=1e-13 * np.abs(q[5:8]).max())
        assert w[8] == q[8]


# ---- O2: fluxes are sqrt(-g) J^d, sqrt(-g) T^d_j, and alpha *F^{kd} -------------
@pytest.mark.parametrize("d", [0, 1, 2])
def test_flux_matches_covariant_definitions(d):
    P, M = states(12 + d, 200)
    for q, m in zip(P, M):
        f = fluid4(q, m, GAM)
        al = m[0]
        T, G, u = f["T"], f["G"], f["u"]
        F = ob.flux_point(d, q, m, GAM, 0)
        w = ob.prim2con_point(q, m, GAM)
        FD = al * q[0] * u[1 + d]                        # alpha rho u^d
        FS = al * (T[1 + d] @ G)[1:]                     # alpha T^d_j
        Ftau = al * al * T[0, 1 + d] - FD                # alpha (alpha T^{0d}) - flux of D
        FB = al * f["Fdual"][1:, 1 + d]                  # alpha *F^{kd}
        sc = np.abs(F[:5]).max() + np.abs(w[:5]).max()
        assert abs(F[0] - FD) <= 1e-12 * sc
        assert np.allclose(F[1:4], FS, rtol=0, atol=1e-12 * sc)
        assert abs(F[4] - Ftau) <= 1e-12 * sc
        assert np.allclose(F[5:8], FB, rtol=0, atol=1e-12 * (np.abs(FB).max() + np.abs(q[5:8]).max()))
        assert F[5 + d] == 0.0 or abs(F[5 + d]) < 1e-16 * np.abs(q[5:8]).max()
        assert F[8] == 0.0


def test_cleaning_flux_rows():
    """R14: with psi = 0 the cleaning rows differ from the plain induction flux only by the
    -beta^k B^d piece that the cleaning source restores; the psi rows are alpha gamma^{kd} psi and
    alpha B^d - beta^d psi (exact eigen-structure checked in test_wavespeeds_bound_jacobian)."""
    P, M = states(15, 100)
    for q, m in zip(P, M):
        gi = np.linalg.inv(gamma3(m))
        for d in range(3):
            q0 = q.copy(); q0[8] = 0.0
            F0 = ob.flux_point(d, q0, m, GAM, 0)
            F1 = ob.flux_point(d, q0, m, GAM, 1)
            assert np.allclose(F1[:5], F0[:5], rtol=0, atol=0)
            for k in range(3):
                assert np.isclose(F1[5 + k] - F0[5 + k], -m[1 + k] * q[5 + d], rtol=1e-11, atol=1e-15)
            Fp = ob.flux_point(d, q, m, GAM, 1)
            for k in range(3):
                assert np.isclose(Fp[5 + k] - F1[5 + k], m[0] * gi[k, d] * q[8], rtol=1e-10, atol=1e-16)
            assert np.isclose(Fp[8], m[0] * q[5 + d] - m[1 + d] * q[8], rtol=1e-12, atol=1e-18)


# ---- O3: wave speeds ----------------------------------------------------------------------------
def _jacobian_eigs(d, q, m, cleaning):
    """Eigenvalues of dF/dU by finite differences of the oracle's flux and prim2con (numpy eig)."""
    # without cleaning B^d is not a wave variable in 1D (its flux row is identically zero): drop it
    idx = list(range(9)) if cleaning else [c for c in range(8) if c != 5 + d]
    n = len(idx)
    A = np.zeros((n, n)); Bm = np.zeros((n, n))
    for k, c in enumerate(idx):
        e = 1e-6 * max(abs(q[c]), 1e-3)
        qp, qm = q.copy(), q.copy()
        qp[c] += e; qm[c] -= e
        A[:, k] = (ob.flux_point(d, qp, m, GAM, cleaning)[idx] - ob.flux_point(d, qm, m, GAM, cleaning)[idx]) / (2 * e)
        Bm[:, k] = (ob.prim2con_point(qp, m, GAM)[idx] - ob.prim2con_point(qm, m, GAM)[idx]) / (2 * e)
    return np.linalg.eigvals(A @ np.linalg.inv(Bm))


def test_wavespeeds_hydro_equal_jacobian_extremes():
    """B = 0: the bound is exact, lambda+- are the extreme eigenvalues of the flux Jacobian."""
    P, M = states(21, 60, vmax=0.9)
    for q, m in zip(P, M):
        q = q.copy(); q[5:9] = 0.0
        q[4] = max(q[4], 1e-2 * q[0])
        for d in range(3):
            lam = ob.wavespeed_point(d, q, m, GAM, 0)
            # hydro sub-system only: D, S, tau rows/cols
            n = 5
            A = np.zeros((n, n)); Bm = np.zeros((n, n))
            for c in range(n):
                e = 1e-6 * max(abs(q[c]), 1e-3)
                qp, qm = q.copy(), q.copy(); qp[c] += e; qm[c] -= e
                A[:, c] = (ob.flux_point(d, qp, m, GAM, 0)[:n] - ob.flux_point(d, qm, m, GAM, 0)[:n]) / (2 * e)
                Bm[:, c] = (ob.prim2con_point(qp, m, GAM)[:n] - ob.prim2con_point(qm, m, GAM)[:n]) / (2 * e)
            ev = np.linalg.eigvals(A @ np.linalg.inv(Bm))
            assert np.abs(ev.imag).max() < 1e-5
            assert np.isclose(ev.real.max(), lam[1], rtol=0, atol=2e-6)
            assert np.isclose(ev.real.min(), lam[0], rtol=0, atol=2e-6)


@pytest.mark.parametrize("cleaning", [0, 1])
def test_wavespeeds_bound_jacobian(cleaning):
    """B != 0: every characteristic speed of the full system lies inside [lambda-, lambda+]
    (PAPER.md:78 'approximate maximal wave speeds'); with cleaning the light cone is included."""
    P, M = states(22, 60, vmax=0.9)
    for q, m in zip(P, M):
        q = q.copy()
        q[4] = max(q[4], 1e-2 * q[0])
        gi = np.linalg.inv(gamma3(m))
        for d in range(3):
            lam = ob.wavespeed_point(d, q, m, GAM, cleaning)
            ev = _jacobian_eigs(d, q, m, cleaning)
            assert ev.real.max() <= lam[1] + 1e-5
            assert ev.real.min() >= lam[0] - 1e-5
            c = m[0] * np.sqrt(gi[d, d])
            # never outside the light cone
            assert lam[1] <= -m[1 + d] + c + 1e-13 and lam[0] >= -m[1 + d] - c - 1e-13
            if cleaning:
                assert np.isclose(ev.real.max(), -m[1 + d] + c, atol=1e-5)
                assert np.isclose(ev.real.min(), -m[1 + d] - c, atol=1e-5)
                assert np.isclose(lam[1], -m[1 + d] + c, rtol=1e-13)


def test_wavespeed_closed_form_limits():
    """P9: flat, B = 0, motion along d: (v +- cs)/(1 +- v cs); a^2 -> 1: -beta^d +- alpha sqrt(gamma^dd)."""
    flat = np.array([1, 0, 0, 0, 1, 0, 0, 1, 0, 1.0])
    for v in [-0.7, 0.0, 0.3, 0.9]:
        W = 1 / np.sqrt(1 - v * v)
        rho, p = 1.0, 0.7
        q = np.array([rho, W * v, 0, 0, p, 0, 0, 0, 0.0])
        h = 1 + GAM / (GAM - 1) * p / rho
        cs = np.sqrt(GAM * p / (rho * h))
        lam = ob.wavespeed_point(0, q, flat, GAM, 0)
        assert np.isclose(lam[1], (v + cs) / (1 + v * cs), rtol=1e-14)
        assert np.isclose(lam[0], (v - cs) / (1 - v * cs), rtol=1e-14)
    P, M = states(23, 20)
    for q, m in zip(P, M):
        q = q.copy(); q[5:8] *= 1e6 / np.sqrt(q[0])  # magnetically dominated: v_A -> 1
        gi = np.linalg.inv(gamma3(m))
        for d in range(3):
            lam = ob.wavespeed_point(d, q, m, GAM, 0)
            c = m[0] * np.sqrt(gi[d, d])
            assert np.isclose(lam[1], -m[1 + d] + c, rtol=1e-6) and np.isclose(lam[0], -m[1 + d] - c, rtol=1e-6)


# ---- O4: MC limiter ------------------------------------------------------------------------------
def test_mc_slope_properties():
    rng = np.random.default_rng(5)
    # exact on linear data, zero at extrema, TVD bound, symmetric under reflection and sign
    assert ob.mc_slope(1.0, 2.0, 3.0) == 1.0
    assert ob.mc_slope(3.0, 1.0, 2.0) == 0.0 and ob.mc_slope(1.0, 1.0, 2.0) == 0.0
    assert ob.mc_slope(0.0, 1.0, 10.0) == 2.0          # limited by 2*|left difference|
    assert ob.mc_slope(0.0, 9.0, 10.0) == 2.0          # limited by 2*|right difference|
    assert ob.mc_slope(0.0, 1.0, 2.5) == 1.25          # central difference inside the bounds
    for _ in range(2000):
        a, b, c = rng.normal(size=3)
        s = ob.mc_slope(a, b, c)
        assert s == -ob.mc_slope(-a, -b, -c)
        assert s == -ob.mc_slope(c, b, a)
        lo, hi = min(a, b, c), max(a, b, c)
        assert lo - 1e-15 <= b + s / 2 <= hi + 1e-15 and lo - 1e-15 <= b - s / 2 <= hi + 1e-15
        assert abs(s) <= 2 * min(abs(b - a), abs(c - b)) + 1e-300


# ---- O5: HLLE ------------------------------------------------------------------------------------
@pytest.mark.parametrize("cleaning", [0, 1])
def test_hlle_consistency_and_upwinding(cleaning):
    P, M = states(31, 100)
    for q, m in zip(P, M):
        sq = np.sqrt(np.linalg.det(gamma3(m)))
        for d in range(3):
            F = ob.flux_point(d, q, m, GAM, cleaning)
            Phi = ob.hlle_point(d, q, q, m, GAM, cleaning)
            assert np.allclose(Phi, sq * F, rtol=1e-12, atol=1e-14 * np.abs(F).max())
    # supersonic flow to the right, no cleaning: pure upwind flux of the left state
    flat = np.array([1, 0, 0, 0, 1, 0, 0, 1, 0, 1.0])
    W = 1 / np.sqrt(1 - 0.99 ** 2)
    qL = np.array([1.0, W * 0.99, 0, 0, 1e-3, 0, 0, 0, 0.0])
    qR = np.array([0.5, W * 0.99, 0, 0, 2e-3, 0, 0, 0, 0.0])
    assert ob.wavespeed_point(0, qL, flat, GAM, 0)[0] > 0
    assert np.allclose(ob.hlle_point(0, qL, qR, flat, GAM, 0), ob.flux_point(0, qL, flat, GAM, 0), rtol=1e-14)


def test_hlle_constant_lapse_rescaling():
    """The alpha-in-HLL slip: with gamma = delta, beta = 0 and constant lapse a, the system is
    flat space with time rescaled by a, so Phi(alpha = a) = a * Phi(alpha = 1) for any L/R pair."""
    P, M = states(32, 100, curved=False)
    P2, _ = states(33, 100, curved=False)
    for qL, qR, m in zip(P, P2, M):
        for a in (0.5, 1.7):
            ma = m.copy(); ma[0] = a
            for cl in (0, 1):
                f1 = ob.hlle_point(0, qL, qR, m, GAM, cl)
                fa = ob.hlle_point(0, qL, qR, ma, GAM, cl)
                assert np.allclose(fa, a * f1, rtol=1e-12, atol=1e-15 * np.abs(f1).max())


# ---- O8: con2prim --------------------------------------------------------------------------------
def test_roundtrip_prim_cons_prim():
    """P1 (north_star): prim -> cons -> prim to 1e-12 for E/p <= 1e3, |v| <= 0.95, random SPD gamma."""
    P, M = states(41, 6000)
    par = OracleParams.default(gamma_ad=GAM)
    nchk = 0
    worst = 0.0
    for q, m in zip(P, M):
        w = ob.prim2con_point(q, m, GAM)
        g = gamma3(m)
        # domain of the pin: the round-trip error is eps * (E/p) * cond(gamma) (the contractions
        # gamma^{ij} S_i S_j and gamma_ij B^i B^j cancel for a nearly degenerate 3-metric)
        if (w[4] + w[0]) / q[4] > 1e3 or np.linalg.cond(g) > 20:
            continue
        rc, q2, it = ob.con2prim_point(w, m, par)   # built-in guess: no help from the answer
        assert rc == 0 and it <= 30
        un = np.sqrt(1 + q[1:4] @ g @ q[1:4])
        err = max(abs(q2[0] - q[0]) / q[0], abs(q2[4] - q[4]) / q[4],
                  np.sqrt((q2[1:4] - q[1:4]) @ g @ (q2[1:4] - q[1:4])) / un)
        worst = max(worst, err)
        assert np.array_equal(q2[5:9], q[5:9])
        nchk += 1
    assert nchk > 3000
    assert worst <= 1e-12, worst


def test_con2prim_root_is_unique_and_matches_bisection():
    """P2: brute-force scan of f(Z) on a fine log grid: exactly one sign change in the admissible
    region (v^2 < 1); bisection there agrees with the Newton result."""
    P, M = states(42, 300)
    par = OracleParams.default(gamma_ad=GAM)
    for q, m in zip(P, M):
        w = ob.prim2con_point(q, m, GAM)
        rc, q2, it = ob.con2prim_point(w, m, par)
        assert rc == 0
        g = gamma3(m)
        W2 = 1 + q2[1:4] @ g @ q2[1:4]
        Znewton = (q2[0] + GAM / (GAM - 1) * q2[4]) * W2
        Zs = Znewton * 1.0007 * np.logspace(-6, 6, 2401)   # offset: the root is not a grid point
        f = np.array([ob.c2p_residual_point(z, w, m, GAM) for z in Zs])
        ok = np.isfinite(f)
        first = np.argmax(ok)
        assert ok[first:].all()          # admissible region is a half line Z > Zmin
        sg = np.sign(f[first:])
        changes = np.nonzero(sg[1:] * sg[:-1] < 0)[0]
        assert len(changes) == 1
        lo, hi = Zs[first + changes[0]], Zs[first + changes[0] + 1]
        flo = ob.c2p_residual_point(lo, w, m, GAM)
        for _ in range(200):
            mid = 0.5 * (lo + hi)
            fm = ob.c2p_residual_point(mid, w, m, GAM)
            if fm * flo > 0:
                lo, flo = mid, fm
            else:
                hi = mid
        # both are roots of the same rounded f: they agree to its noise level eps*cond(gamma)/f'
        assert abs(0.5 * (lo + hi) - Znewton) <= 1e-14 * max(np.linalg.cond(g), 10) ** 2 * Znewton


def test_con2prim_guess_independence_and_failure():
    P, M = states(43, 200)
    par = OracleParams.default(gamma_ad=GAM)
    for q, m in zip(P, M):
        w = ob.prim2con_point(q, m, GAM)
        rc1, a, _ = ob.con2prim_point(w, m, par, -1.0)
        Z = (q[0] + GAM / (GAM - 1) * q[4]) * (1 + q[1:4] @ gamma3(m) @ q[1:4])
        rc2, b, it2 = ob.con2prim_point(w, m, par, Z * 3.0)
        rc3, c, it3 = ob.con2prim_point(w, m, par, Z)
        assert rc1 == rc2 == rc3 == 0 and it3 <= 2
        E_over_p = (w[4] + w[0]) / q[4]
        tol = 1e-14 * max(E_over_p, 100)
        assert np.allclose(a, b, rtol=tol, atol=1e-300) and np.allclose(a, c, rtol=tol, atol=1e-300)
    # unphysical input (negative D, NaN) must be reported, not returned
    w = np.array([-1.0, 0, 0, 0, 1.0, 0, 0, 0, 0]); flat = np.array([1, 0, 0, 0, 1, 0, 0, 1, 0, 1.0])
    assert ob.con2prim_point(w, flat, par)[0] == 1
    w = np.array([1.0, np.nan, 0, 0, 1.0, 0, 0, 0, 0])
    assert ob.con2prim_point(w, flat, par)[0] == 1


# ---- O8b: the two-unknown scheme (reading R10b) ----------------------------------------
def test_two_unknown_scheme_roundtrip_and_agreement_with_the_one_unknown_scheme():
    """The physical root is unique, so Newton on (Z, v^2) must return the primitives Newton on Z returns
    (two different iterations, one answer), and it must pass the P1 round trip on its own: 1e-12 for
    E/p <= 1e3.  Both start from the built-in guess."""
    P, M = states(43, 4000)
    par1 = OracleParams.default(gamma_ad=GAM)
    par2 = OracleParams.default(gamma_ad=GAM, c2p_scheme=1)
    nchk, worst_rt, worst_ag = 0, 0.0, 0.0
    for q, m in zip(P, M):
        w = ob.prim2con_point(q, m, GAM)
        g = gamma3(m)
        if (w[4] + w[0]) / q[4] > 1e3 or np.linalg.cond(g) > 20:
            continue
        rc1, a, it1 = ob.con2prim_point(w, m, par1)
        rc2, b, it2 = ob.con2prim_point(w, m, par2)
        assert rc1 == 0 and rc2 == 0 and it2 <= 30, (rc1, rc2, it2)
        un = np.sqrt(1 + q[1:4] @ g @ q[1:4])
        dist = lambda x, y: max(abs(x[0] - y[0]) / y[0], abs(x[4] - y[4]) / y[4],
                                np.sqrt((x[1:4] - y[1:4]) @ g @ (x[1:4] - y[1:4])) / un)
        worst_rt = max(worst_rt, dist(b, q))
        worst_ag = max(worst_ag, dist(b, a))
        assert np.array_equal(b[5:9], q[5:9])
        nchk += 1
    assert nchk > 2000
    assert worst_rt <= 1e-12, worst_rt
    assert worst_ag <= 1e-12, worst_ag


def test_two_unknown_scheme_is_a_different_iteration():
    """Guard against the second scheme silently calling the first: from a poor guess the two take
    different numbers of steps on some states."""
    P, M = states(44, 300)
    par1 = OracleParams.default(gamma_ad=GAM)
    par2 = OracleParams.default(gamma_ad=GAM, c2p_scheme=1)
    differ = 0
    for q, m in zip(P, M):
        w = ob.prim2con_point(q, m, GAM)
        it1 = ob.con2prim_point(w, m, par1)[2]
        it2 = ob.con2prim_point(w, m, par2)[2]
        differ += it1 != it2
    assert differ > 30, differ


# ---- O4b: PPM edge values (reading R5b) ---------------------------------------------------
def test_ppm_edges_closed_forms():
    """Pins of the piecewise parabolic reconstruction: exact on linear data; the unlimited interface value
    a_{i+1/2} = q_i + (q_{i+1} - q_i)/2 - (d_{i+1} - d_i)/6 when no slope is clipped; flat at a local extremum;
    edges bounded by the three cells they come from; and Colella & Woodward's no-interior-extremum condition
    |aR - aL| >= 6 |q0 - (aL + aR)/2| after limiting."""
    # linear data: edges are the linear interpolants
    for slope in (0.3, -2.0):
        q5 = [1.0 + slope * i for i in range(-2, 3)]
        aL, aR = ob.ppm_edges(q5)
        assert abs(aL - (1.0 - slope / 2)) < 1e-15 and abs(aR - (1.0 + slope / 2)) < 1e-15
    # unlimited interface value: (7 (q_i + q_{i+1}) - (q_{i-1} + q_{i+2})) / 12 when no slope is clipped
    q5 = [0.0, 1.0, 2.1, 3.3, 4.6]                 # monotone, gently curved: MC slopes are the centred ones
    aL, aR = ob.ppm_edges(q5)
    # slopes: d_{-1} = (2.1 - 0)/2, d_0 = (3.3 - 1)/2, d_1 = (4.6 - 2.1)/2
    dm, d0, dp = 1.05, 1.15, 1.25
    assert abs(aL - (1.0 + 0.55 - (d0 - dm) / 6)) < 1e-15
    assert abs(aR - (2.1 + 0.6 - (dp - d0) / 6)) < 1e-15
    # local extremum: flat
    assert ob.ppm_edges([0.0, 1.0, 2.0, 1.0, 0.0]) == (2.0, 2.0)
    # steep one-sided profile: the parabola would overshoot, the monotonisation pulls one edge in
    aL, aR = ob.ppm_edges([0.0, 0.0, 0.1, 1.0, 1.0])
    assert 0.0 <= aL <= 0.1 <= aR <= 1.0
    # the parabola through (aL, q0 as mean, aR) has no interior extremum after limiting:
    # |aR - aL| >= 6 |q0 - (aL + aR)/2|  (Colella & Woodward's condition)
    rng = np.random.default_rng(7)
    for _ in range(2000):
        q5 = rng.normal(size=5).cumsum() if rng.random() < 0.5 else rng.normal(size=5)
        aL, aR = ob.ppm_edges(q5)
        lo, hi = min(q5[1:4]), max(q5[1:4])
        assert lo - 1e-14 <= aL <= hi + 1e-14 and lo - 1e-14 <= aR <= hi + 1e-14
        assert abs(aR - aL) * (1 + 1e-12) + 1e-15 >= 6 * abs(q5[2] - 0.5 * (aL + aR))
