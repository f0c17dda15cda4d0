"""Shared helpers of the GPU-vs-oracle parity tests (the parity bar)."""
import numpy as np

FIELDS = ["rho", "vx", "vy", "vz", "p", "Bx", "By", "Bz"]


def rel_l1(gpu, ora):
    """Per-field relative L1 = sum|gpu - ora| / sum|ora| over interior cells (BASELINE.json north_star).

    A field that is identically zero in the oracle is compared by absolute max against the scale of
    its vector (v or B), as SURVEY.md 8(d) prescribes; the returned number is then max|diff|/scale.
    """
    gpu = np.asarray(gpu, dtype=np.float64)
    ora = np.asarray(ora, dtype=np.float64)
    out = {}
    for f, name in enumerate(FIELDS):
        den = np.abs(ora[f]).sum()
        num = np.abs(gpu[f] - ora[f]).sum()
        if den > 0:
            out[name] = num / den
        else:
            grp = slice(1, 4) if 1 <= f <= 3 else (slice(5, 8) if f >= 5 else slice(f, f + 1))
            scale = np.abs(ora[grp]).max()
            out[name] = np.abs(gpu[f] - ora[f]).max() / (scale if scale > 0 else 1.0)
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
