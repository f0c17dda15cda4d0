"""Shared helpers of the GPU-vs-oracle parity tests (the parity bar)."""
import numpy as np

FIELDS = ["rho", "vx", "vy", "vz", "p", "Bx", "By", "Bz"]


GROUP_FLOOR = 1e-2


def rel_l1(gpu, ora):
    """Per-field relative L1 = sum|gpu - ora| / sum|ora| over interior cells (BASELINE.json north_star).

    Reading: for a component of v or B the denominator is not allowed to fall
    below GROUP_FLOOR (1 %) of the largest component's L1 norm of the same vector.  A component that a
    symmetry keeps at truncation level (v^x of a transverse wave, v^z of a star rotating about z) or
    exactly zero (B^z of config 1) has no scale of its own: its round-off error is set by the size of
    the vector, in any implementation, so that is what it is measured against.
    """
    gpu = np.asarray(gpu, dtype=np.float64)
    ora = np.asarray(ora, dtype=np.float64)
    norms = [np.abs(ora[f]).sum() for f in range(len(FIELDS))]
    out = {}
    for f, name in enumerate(FIELDS):
        grp = range(1, 4) if 1 <= f <= 3 else (range(5, 8) if f >= 5 else range(f, f + 1))
        den = max(norms[f], GROUP_FLOOR * max(norms[g] for g in grp))
        num = np.abs(gpu[f] - ora[f]).sum()
        out[name] = num / den if den > 0 else (0.0 if num == 0 else np.inf)
    return out


def oracle_for(w, **par_over):
    from oracle import Oracle, OracleParams
    par = OracleParams.default(**{**w.params, **par_over})
    o = Oracle(w.n, w.h, w.bc, par)
    o.set_metric(w.alpha, w.beta3, w.gamma6)
    o.set_primitives(w.prim8)
    return o


def assert_parity(gpu, ora, tol, what=""):
    r = rel_l1(gpu, ora)
    bad = {k: v for k, v in r.items() if not (v <= tol)}
    assert not bad, f"{what}: rel L1 above {tol:g}: {bad} (all: {r})"
    return r
