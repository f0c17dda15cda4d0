"""BASELINE.json's five configs at their STATED sizes against the oracle (pytest -m gpu), the rows VERDICT round 1
found compared only at reduced sizes: config 4 (the star, 192^3), config 2 (Alfven wave, 64^3 and the 32/64/128
convergence check on the GPU output), config 5 at 384^3, and the degenerate branches of the recovery (failure,
reset to atmosphere with the ambient medium at the floor).  Tolerances are north_star's (tests/test_gpu_parity.py).

The oracle runs 4-5e6 zone-updates/s on 16 host cores, so the full 501 substeps of config 4 at 192^3 take about
a quarter of an hour; the default length here is 60 full steps (180 substeps, 3.4e8 atmosphere resets), and
HZ_LONG_TESTS=1 runs all 167 (profiles/r02_fullruns.md records that run)."""
import dataclasses
import os

import numpy as np
import pytest

import workloads as wl
from parity import assert_parity, floor_flip_mask, oracle_for
from test_gpu_parity import TOL32_SUB, TOL64_RUN, TOL64_SUB, horizon, sub_block

pytestmark = pytest.mark.gpu
LONG = os.environ.get("HZ_LONG_TESTS", "0") == "1"


def _counts_equal(do, dg, keys=("c2p_fail", "atm_reset", "p_floor")):
    for k in keys:
        assert do[k] == dg[k], (k, do[k], dg[k])


def test_config4_star_192_run_fp64():
    """BASELINE config 4 at its own 192^3 (the star on a fixed curved metric).  93 % of
    the cells are atmosphere and are reset in every substep -- the branch most likely to drift between CPU and
    GPU -- so the reset, floor and failure counts must be identical and every cell within 1e-7."""
    w = wl.tov_star(192)
    nsteps = w.nsteps if LONG else 60
    o = oracle_for(w)
    hz = horizon(w, "f64")
    hz.step(w.dt, nsteps)          # asynchronous: the GPU run is over long before the oracle's
    o.step(w.dt, nsteps)
    got, ref = hz.get_primitives(), o.get_primitives()
    assert np.isfinite(got).all()
    r = assert_parity(got, ref, TOL64_RUN, f"star 192^3, {nsteps} steps ({3 * nsteps} substeps) fp64")
    do, dg = o.diagnostics(), hz.diagnostics()
    assert do["atm_reset"] > 1e8
    _counts_equal(do, dg)
    for k in ("sumD", "sumTau"):
        assert abs(do[k] - dg[k]) <= 1e-9 * abs(do[k]), (k, do[k], dg[k])
    print("star 192^3 max rel L1", max(r.values()), "resets", dg["atm_reset"], "p floors", dg["p_floor"])
    hz.close()


@pytest.mark.parametrize("dtype", ["f32", "f32h"])
def test_config4_star_192_one_substep_fp32_and_mixed(dtype):
    w = wl.tov_star(192)
    o = oracle_for(w)
    hz = horizon(w, dtype)
    o.substeps(w.dt, 1)
    hz.substeps(w.dt, 1)
    got, ref = hz.get_primitives(), o.get_primitives()
    flips = floor_flip_mask(got, ref, w.params["rho_atm"], w.params["atm_tol"])
    assert flips.sum() <= 2e-4 * w.ncell, f"{flips.sum()} atmosphere-branch flips"
    assert_parity(got, ref, TOL32_SUB, f"star 192^3 {dtype} 1 substep", mask=flips)
    assert hz.diagnostics()["c2p_fail"] == 0
    hz.close()


def test_config2_alfven_64_one_period_fp64():
    """BASELINE config 2 at its own 64^3: one crossing time (387 steps = 1161 substeps) against the oracle."""
    w = wl.alfven_wave(64)
    o = oracle_for(w)
    hz = horizon(w, "f64")
    hz.step(w.dt, w.nsteps)
    o.step(w.dt, w.nsteps)
    assert_parity(hz.get_primitives(), o.get_primitives(), TOL64_RUN, f"alfven 64^3, {w.nsteps} steps fp64")
    _counts_equal(o.diagnostics(), hz.diagnostics())
    hz.close()


def test_config2_convergence_order_measured_on_the_gpu():
    """BASELINE config 2's convergence check, on the GPU output: the circularly polarised wave is an exact
    solution, so after one period the fields must be back on the initial data; the L1 error of
    the transverse components at 32^3 / 64^3 / 128^3 must fall by at least 2^1.7 per doubling (MC clips the
    extrema, so the formal order 2 is not reached)."""
    errs = []
    for n in (32, 64, 128):
        w = wl.alfven_wave(n)
        hz = horizon(w, "f64")
        hz.step(w.dt, w.nsteps)
        p = hz.get_primitives()
        d = hz.diagnostics()
        assert d["c2p_fail"] == 0 and d["atm_reset"] == 0
        errs.append(max(np.abs(p[q] - w.prim8[q]).mean() for q in (1, 2, 3, 5, 6, 7)))
        hz.close()
    o1, o2 = np.log2(errs[0] / errs[1]), np.log2(errs[1] / errs[2])
    print("alfven L1 errors at 32/64/128:", errs, "orders", o1, o2)
    assert o1 > 1.7 and o2 > 1.7, (errs, o1, o2)


@pytest.mark.parametrize("dtype,tol", [("f64", TOL64_SUB * 10), ("f32", TOL32_SUB * 3), ("f32h", TOL32_SUB * 3)])
def test_config5_sampled_blocks_384(dtype, tol):
    """BASELINE config 5 at its largest grid, 384^3 (20.8 GB of state in fp64), in the launch configuration the
    bench uses: one full RK3 step, compared cell by cell with the oracle run on 44^3 sub-blocks of the same
    inputs (a cell depends only on cells within 9 zones of it after three substeps; the bar
    after three substeps is 10x / 3x the one-substep bar)."""
    w = wl.kerr_sweep(384)
    hz = horizon(w, dtype)
    hz.step(w.dt, 1)
    got = hz.get_primitives()
    assert np.isfinite(got).all()
    m = 12
    for (k0, j0, i0) in [(0, 0, 0), (340, 340, 340), (170, 201, 333), (301, 12, 150)]:
        sl = (slice(k0, k0 + 44), slice(j0, j0 + 44), slice(i0, i0 + 44))
        ws = sub_block(w, sl)
        o = oracle_for(ws)
        o.step(w.dt, 1)
        ref = o.get_primitives()
        lo = [0 if s.start == 0 else m for s in sl]                    # a true domain boundary needs no margin
        hi = [44 if s.stop == 384 else 44 - m for s in sl]
        inner = tuple(slice(a, b) for a, b in zip(lo, hi))
        g = got[(slice(None),) + sl][(slice(None),) + inner]
        assert_parity(g, ref[(slice(None),) + inner], tol, f"384^3 {dtype} block at {(k0, j0, i0)}")
    hz.close()


def _same_outcome_despite_failure_flags(o, hz, w, what):
    """What must agree in a run with failing recoveries.  A recovery "fails" here when its Newton step stalls
    just above 1e-13 Z in a cell at atmosphere level (R11 measures the step against Z alone; the round-off of the
    residual is eps (Z + B^2)): whether it stalls above or below the tolerance depends on rounding order, so the
    FLAG may differ between CPU and GPU in a few cells -- but such a cell is reset to atmosphere either way (as
    a failure, or as rho < rho_atm (1 + atm_tol)), so the reset count, the set of atmosphere cells and every
    field must agree.  Measured (profiles/r02_fullruns.md): identical resets and fields to 1e-14 while the
    failure flags differ by up to 10 %."""
    do, dg = o.diagnostics(), hz.diagnostics()
    assert do["c2p_fail"] > 0 and dg["c2p_fail"] > 0, (do["c2p_fail"], dg["c2p_fail"])
    for k in ("atm_reset", "p_floor", "c2p_maxit_seen"):
        assert do[k] == dg[k], (k, do[k], dg[k])
    assert 0.4 * do["c2p_fail"] <= dg["c2p_fail"] <= 2.5 * do["c2p_fail"], (do["c2p_fail"], dg["c2p_fail"])
    got, ref = hz.get_primitives(), o.get_primitives()
    atm = ref[0] == w.params["rho_atm"]
    assert np.array_equal(got[0] == w.params["rho_atm"], atm)
    assert np.all(got[1:4][:, atm] == 0)
    print(f"{what}: failed recoveries oracle {do['c2p_fail']} / GPU {dg['c2p_fail']}, resets {dg['atm_reset']} on both")
    assert_parity(got, ref, TOL64_RUN, what)


def test_recovery_failures_match_the_oracle():
    """The fragile step: a run in which the primitive recovery FAILS.  The blast of config 3
    on a 32^3 copy: once the wave has reached the zero-gradient boundaries the strongly magnetised, nearly
    evacuated ambient medium drives recoveries to failure (first failures between steps 66 and 80 on both
    sides).  Up to step 65 (4 992 resets, 128 pressure floors, no failure): identical counts and every cell within
    1e-7.  At step 90 (2 304 failures in the oracle, 72 448 resets): see _same_outcome_despite_failure_flags.
    (Beyond step 90 the two runs part for good: a reset that happens on one side only changes its neighbours.)"""
    w = wl.blast(32)
    o = oracle_for(w)
    hz = horizon(w, "f64")
    o.step(w.dt, 65)
    hz.step(w.dt, 65)
    do, dg = o.diagnostics(), hz.diagnostics()
    assert do["c2p_fail"] == 0 and do["atm_reset"] > 1000 and do["p_floor"] > 0
    _counts_equal(do, dg, ("c2p_fail", "atm_reset", "p_floor", "c2p_maxit_seen"))
    assert_parity(hz.get_primitives(), o.get_primitives(), TOL64_RUN, "blast 32^3, 65 steps (before the first failure)")
    o.step(w.dt, 25)
    hz.step(w.dt, 25)
    _same_outcome_despite_failure_flags(o, hz, w, "blast 32^3, 90 steps")
    hz.close()


def test_failed_recovery_resets_to_atmosphere_like_the_oracle():
    """Degenerate case of the method (the case VERDICT round 1 asked to be put back): the blast with its ambient
    medium right at the floor, so that a state that evacuates a cell ends in the atmosphere branch -- 12 480 cells
    are reset in every substep and, from the fifth substep on, some of their recoveries fail outright."""
    w = wl.blast(24)
    prim = w.prim8.copy()
    prim[0] = np.where(prim[0] < 5e-3, 1.0000005e-7, prim[0])
    w = dataclasses.replace(w, prim8=prim)
    o = oracle_for(w)
    hz = horizon(w)
    o.substeps(w.dt, 4)
    hz.substeps(w.dt, 4)
    do, dg = o.diagnostics(), hz.diagnostics()
    assert do["atm_reset"] > 0 and do["c2p_fail"] == 0
    _counts_equal(do, dg, ("c2p_fail", "atm_reset", "p_floor", "c2p_maxit_seen"))
    assert_parity(hz.get_primitives(), o.get_primitives(), TOL64_RUN, "blast with the ambient medium at the floor, 4 substeps")
    o.substeps(w.dt, 5)
    hz.substeps(w.dt, 5)
    _same_outcome_despite_failure_flags(o, hz, w, "blast with the ambient medium at the floor, 3 steps")
    hz.close()
