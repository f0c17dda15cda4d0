"""GPU-vs-oracle parity through the C-ABI (pytest -m gpu).  Tolerances are BASELINE.json's north_star:
fp64 rel. L1 <= 1e-10 per field after one substep and <= 1e-7 after the full run; fp32 <= 1e-4 after one
substep against the fp64 oracle.  Inputs come from workloads/ (seeded, synthetic); expected values come
from oracle/ only."""
import dataclasses

import numpy as np
import pytest

import workloads as wl
from parity import assert_parity, floor_flip_mask, oracle_for, rel_l1

pytestmark = pytest.mark.gpu

TOL64_SUB, TOL64_RUN, TOL32_SUB = 1e-10, 1e-7, 1e-4


def horizon(w, dtype="f64", **kw):
    from paper_1102_5202_b200 import Horizon
    return Horizon.from_workload(w, dtype=dtype, **kw)


def sub_block(w, sl):
    """The workload restricted to the index block sl = (kslice, jslice, islice)."""
    f = lambda a: np.ascontiguousarray(a[(slice(None),) + sl]) if a.ndim == 4 else np.ascontiguousarray(a[sl])
    n = tuple(s.stop - s.start for s in sl[::-1])
    return dataclasses.replace(w, n=n, alpha=f(w.alpha), beta3=f(w.beta3), gamma6=f(w.gamma6), prim8=f(w.prim8))


# sizes span several thread blocks / tiles and leave ragged tails in every axis
SMALL = {
    "tube_x": lambda: wl.shock_tube(400, axis=0),
    "tube_x_ragged": lambda: wl.shock_tube(403, axis=0),
    "tube_y": lambda: wl.shock_tube(131, axis=1),
    "tube_z": lambda: wl.shock_tube(77, axis=2),
    "alfven_3d": lambda: wl.alfven_wave(n=(37, 21, 13)),
    "alfven_2d": lambda: wl.alfven_wave(n=(45, 19, 1)),
    "alfven_1d": lambda: wl.alfven_wave(64, direction="x"),
    "blast": lambda: wl.blast(35),
    "tov": lambda: wl.tov_star(44),
    "kerr": lambda: wl.kerr_sweep(41),
}


@pytest.mark.parametrize("name", sorted(SMALL))
@pytest.mark.parametrize("nsub", [1, 3])
def test_substep_parity_fp64(name, nsub):
    w = SMALL[name]()
    o = oracle_for(w)
    hz = horizon(w, "f64")
    o.substeps(w.dt, nsub)
    hz.substeps(w.dt, nsub)
    assert_parity(hz.get_primitives(), o.get_primitives(), TOL64_SUB, f"{name} fp64 {nsub} substeps")
    # cleaning scalar and densitised conserved variables too
    psi_o, psi_g = o.get_psi(), hz.get_psi()
    assert np.abs(psi_g - psi_o).sum() <= TOL64_SUB * max(np.abs(psi_o).sum(), 1e-300) + 1e-25
    Uo, Ug = o.get_conserved(), hz.get_conserved()
    for q in range(9):
        den = np.abs(Uo[q]).sum()
        scale = den if den > 0 else np.abs(Uo).max() * Uo[q].size
        assert np.abs(Ug[q] - Uo[q]).sum() <= TOL64_SUB * scale, (name, q)
    hz.close()


@pytest.mark.parametrize("name", sorted(SMALL))
def test_substep_parity_fp32(name):
    w = SMALL[name]()
    o = oracle_for(w)
    hz = horizon(w, "f32")
    o.substeps(w.dt, 1)
    hz.substeps(w.dt, 1)
    got = hz.get_primitives()
    assert got.dtype == np.float32
    ref = o.get_primitives()
    flips = floor_flip_mask(got, ref, w.params["rho_atm"], w.params["atm_tol"])
    assert flips.sum() <= 2e-4 * w.ncell, f"{flips.sum()} atmosphere-branch flips"
    assert_parity(got, ref, TOL32_SUB, f"{name} fp32 1 substep", mask=flips)
    hz.close()


@pytest.mark.parametrize("name", sorted(SMALL))
def test_substep_parity_mixed_precision(name):
    """The paper's mixed mode: fp32 storage and face fluxes, fp64 flux
    difference, RK combine and con2prim.  Same bar as pure fp32 against the fp64 oracle."""
    w = SMALL[name]()
    o = oracle_for(w)
    hz = horizon(w, "f32h")
    o.substeps(w.dt, 1)
    hz.substeps(w.dt, 1)
    got = hz.get_primitives()
    assert got.dtype == np.float32
    ref = o.get_primitives()
    flips = floor_flip_mask(got, ref, w.params["rho_atm"], w.params["atm_tol"])
    assert flips.sum() <= 2e-4 * w.ncell, f"{flips.sum()} atmosphere-branch flips"
    assert_parity(got, ref, TOL32_SUB, f"{name} mixed 1 substep", mask=flips)
    hz.close()


def test_mixed_precision_recovers_pressure_better_than_pure_fp32_on_the_star():
    """Why the paper proposes fp64 islands: in fp32 the recovery of p from
    tau + D loses digits where p << rho (the star's envelope and atmosphere, config 4).  After a full
    RK3 step the pressure error of the mixed mode against the fp64 oracle must not exceed pure fp32's,
    and the recovery must never fail in either."""
    w = wl.tov_star(44)
    o = oracle_for(w)
    o.substeps(w.dt, 3)
    ref = o.get_primitives()
    err = {}
    for dt in ("f32", "f32h"):
        hz = horizon(w, dt)
        hz.substeps(w.dt, 3)
        got = hz.get_primitives().astype(np.float64)
        d = hz.diagnostics()
        assert d["c2p_fail"] == 0
        err[dt] = rel_l1(got, ref)
        hz.close()
    assert err["f32h"]["p"] <= err["f32"]["p"] * 1.05, err
    assert err["f32h"]["rho"] <= err["f32"]["rho"] * 1.05, err


def test_full_run_config1_tube_fp64():
    """BASELINE config 1 exactly: 400 cells, CFL 0.4, 400 steps to t = 0.4."""
    w = wl.shock_tube(400)
    assert w.nsteps == 400
    o = oracle_for(w)
    hz = horizon(w, "f64")
    o.step(w.dt, w.nsteps)
    hz.step(w.dt, w.nsteps)
    r = assert_parity(hz.get_primitives(), o.get_primitives(), TOL64_RUN, "tube full run")
    assert max(r.values()) < 1e-9  # in practice round-off level
    do, dg = o.diagnostics(), hz.diagnostics()
    for k in ("c2p_fail", "atm_reset", "p_floor"):
        assert do[k] == dg[k] == 0
    hz.close()


@pytest.mark.parametrize("name,make,nsteps", [
    ("alfven32", lambda: wl.alfven_wave(32), None),          # config 2 at its smallest grid, one period
    ("blast40", lambda: wl.blast(40), 20),                   # config 3 shape, 60 substeps
    ("tov48", lambda: wl.tov_star(48), 12),                  # config 4 shape, 36 substeps
    ("kerr40", lambda: wl.kerr_sweep(40), 34),               # config 5 shape, its full 102 substeps
])
def test_full_run_parity_fp64(name, make, nsteps):
    w = make()
    nsteps = nsteps or w.nsteps
    o = oracle_for(w)
    hz = horizon(w, "f64")
    o.step(w.dt, nsteps)
    hz.step(w.dt, nsteps)
    assert_parity(hz.get_primitives(), o.get_primitives(), TOL64_RUN, f"{name} {nsteps} steps")
    do, dg = o.diagnostics(), hz.diagnostics()
    for k in ("c2p_fail", "atm_reset", "p_floor", "c2p_maxit_seen"):
        assert do[k] == dg[k], (k, do[k], dg[k])
    hz.close()


@pytest.mark.parametrize("name,make", [
    ("blast128", lambda: wl.blast(128)),        # BASELINE config 3 exactly: 128^3, 67 steps = 201 substeps
    ("kerr128", lambda: wl.kerr_sweep(128)),    # BASELINE config 5 at 128^3: 34 steps = 102 substeps
])
def test_full_run_parity_at_baseline_size_fp64(name, make):
    """Full-length runs at BASELINE.json's own sizes against the oracle (about two minutes of oracle time on
    16 host cores): every cell, rel. L1 <= 1e-7 per field, identical floor and failure counts."""
    w = make()
    o = oracle_for(w)
    hz = horizon(w, "f64")
    hz.step(w.dt, w.nsteps)
    o.step(w.dt, w.nsteps)
    got = hz.get_primitives()
    assert np.isfinite(got).all()
    r = assert_parity(got, o.get_primitives(), TOL64_RUN, f"{name} {w.nsteps} steps")
    do, dg = o.diagnostics(), hz.diagnostics()
    for k in ("c2p_fail", "atm_reset", "p_floor"):
        assert do[k] == dg[k], (k, do[k], dg[k])
    for k in ("sumD", "sumTau"):
        assert abs(do[k] - dg[k]) <= 1e-9 * abs(do[k]), (k, do[k], dg[k])
    print(name, "max rel L1", max(r.values()))
    hz.close()


def test_diagnostics_match_oracle():
    w = wl.kerr_sweep(33)
    o = oracle_for(w)
    hz = horizon(w, "f64")
    o.substeps(w.dt, 2)
    hz.substeps(w.dt, 2)
    do, dg = o.diagnostics(), hz.diagnostics()
    for k in ("sumD", "sumSx", "sumSy", "sumSz", "sumTau", "sumBx", "sumBy", "sumBz", "divB_L1"):
        assert abs(dg[k] - do[k]) <= 1e-12 * max(abs(do[k]), 1e-3), (k, dg[k], do[k])  # summation order (R21)
    for k in ("divB_max", "max_speed_over_dx"):
        assert abs(dg[k] - do[k]) <= 1e-11 * abs(do[k]), (k, dg[k], do[k])
    hz.close()


@pytest.mark.parametrize("dtype,tol", [("f64", TOL64_SUB * 10), ("f32", TOL32_SUB * 3), ("f32h", TOL32_SUB * 3)])
def test_bench_configuration_sampled_block_256(dtype, tol):
    """BASELINE config 5 at the bench size (256^3, the launch configuration bench.py times), all three modes:
    after one full RK3 step a cell depends only on cells within 3 x 3 zones of it (two for the MC
    stencil, one for the source differences, per substep), so the oracle run on a 44^3 sub-block of the
    same inputs fixes the inner 20^3 cells one by one."""
    w = wl.kerr_sweep(256)
    hz = horizon(w, dtype)
    hz.step(w.dt, 1)
    got = hz.get_primitives()
    assert np.isfinite(got).all()
    m = 12
    for (k0, j0, i0) in [(0, 0, 0), (106, 117, 90), (212, 212, 212), (31, 200, 140)]:
        sl = (slice(k0, k0 + 44), slice(j0, j0 + 44), slice(i0, i0 + 44))
        ws = sub_block(w, sl)
        o = oracle_for(ws)
        o.step(w.dt, 1)
        ref = o.get_primitives()
        lo = [0 if s.start == 0 else m for s in sl]          # a true domain boundary needs no margin
        inner = tuple(slice(a, 44 - m) for a in lo)
        g = got[(slice(None),) + sl][(slice(None),) + inner]
        assert_parity(g, ref[(slice(None),) + inner], tol, f"256^3 {dtype} block at {(k0, j0, i0)}")
    hz.close()


def test_device_pointers_and_user_buffer_agree_with_host_path():
    import torch
    from paper_1102_5202_b200 import Horizon, HzParams
    w = wl.kerr_sweep(24)
    a = horizon(w, "f64")                       # host numpy inputs, torch-owned state buffer
    par = HzParams.default(**w.params)
    b = Horizon(w.n, w.h, w.bc, dtype="f64", params=par, use_torch_memory=False)  # cudaMalloc'd state
    dev = lambda x: torch.from_numpy(np.ascontiguousarray(x)).cuda()
    b.set_metric(dev(w.alpha), dev(w.beta3), dev(w.gamma6))
    b.set_primitives(dev(w.prim8))
    s = torch.cuda.Stream()
    b.set_stream(s)
    a.step(w.dt, 1)
    b.step(w.dt, 1)
    out = torch.empty((8,) + w.alpha.shape, dtype=torch.float64, device="cuda")
    b.get_primitives(out=out)
    assert np.array_equal(a.get_primitives(), out.cpu().numpy())  # deterministic per cell: bitwise equal
    a.close(); b.close()


def test_bitwise_reproducible():
    w = wl.blast(32)
    outs = []
    for _ in range(2):
        hz = horizon(w, "f32")
        hz.step(w.dt, 2)
        outs.append(hz.get_primitives())
        hz.close()
    assert np.array_equal(outs[0], outs[1])


def test_step_graph_replay_equals_plain_launches_bitwise():
    """hz_step(dt, n >= 2) replays pairs of steps as one CUDA graph (include/hz.h): same kernels, same order, so
    the state after 5 steps equals 15 plain substeps bit for bit, the launch count is the same, and a second call
    (buffer roles swapped by the odd step) is right as well."""
    w = wl.kerr_sweep(20)
    a, b = horizon(w, "f64"), horizon(w, "f64")
    n0 = a.launch_count()
    a.step(w.dt, 5)
    b.substeps(w.dt, 15)
    assert a.launch_count() - n0 == 15
    assert np.array_equal(a.get_primitives(), b.get_primitives())
    a.step(w.dt, 4)
    b.substeps(w.dt, 12)
    assert np.array_equal(a.get_primitives(), b.get_primitives())
    assert np.array_equal(a.get_conserved(), b.get_conserved())
    da, db = a.diagnostics(), b.diagnostics()
    assert da["atm_reset"] == db["atm_reset"] and da["c2p_maxit_seen"] == db["c2p_maxit_seen"]
    a.close(); b.close()


def test_uniform_state_on_constant_curved_metric_is_a_fixed_point():
    n = (20, 12, 9)
    alpha, beta3, gamma6 = wl.constant_metric(n)
    prim = np.zeros((8, n[2], n[1], n[0]))
    prim[0], prim[4] = 1.0, 0.3
    prim[1], prim[2], prim[3] = 0.2, -0.1, 0.05
    prim[5], prim[6], prim[7] = 0.3, 0.1, -0.2
    from paper_1102_5202_b200 import Horizon, HzParams
    hz = Horizon(n, (0.1, 0.1, 0.1), (0, 0, 0), params=HzParams.default(gamma_ad=5.0 / 3.0))
    hz.set_metric(alpha, beta3, gamma6)
    hz.set_primitives(prim)
    hz.step(0.02, 5)
    out = hz.get_primitives()
    assert np.abs(out - prim).max() < 1e-13
    hz.close()


def test_minimum_extent_and_two_cell_axes():
    # 2 cells along y and z (the smallest active extent), ragged x
    w = wl.alfven_wave(n=(19, 2, 2))
    o = oracle_for(w)
    hz = horizon(w)
    o.substeps(w.dt, 3)
    hz.substeps(w.dt, 3)
    assert_parity(hz.get_primitives(), o.get_primitives(), TOL64_SUB, "19x2x2")
    hz.close()
    # a single cell: nothing to sweep, the state must not change
    from paper_1102_5202_b200 import Horizon
    hz = Horizon((1, 1, 1), (1, 1, 1), (0, 0, 0))
    a, b, g = wl.minkowski((1, 1, 1))
    hz.set_metric(a, b, g)
    p = np.array([1.0, 0.1, 0.2, -0.3, 2.0, 0.5, 0.1, 0.2]).reshape(8, 1, 1, 1)
    hz.set_primitives(p)
    hz.step(0.1, 2)
    assert np.abs(hz.get_primitives() - p).max() < 1e-14
    hz.close()


def test_floor_branches_match_the_oracle():
    """Degenerate cases of the method: the atmosphere reset and the pressure floor (R11).
    The star's exterior is atmosphere, so both branches fire in every substep; the counts and the
    fields must agree with the oracle."""
    w = wl.tov_star(40)
    o = oracle_for(w)
    hz = horizon(w)
    o.substeps(w.dt, 4)
    hz.substeps(w.dt, 4)
    do, dg = o.diagnostics(), hz.diagnostics()
    assert do["atm_reset"] > 1000 and do["p_floor"] > 100
    for k in ("c2p_fail", "atm_reset", "p_floor", "c2p_maxit_seen"):
        assert dg[k] == do[k], (k, dg[k], do[k])
    got, ref = hz.get_primitives(), o.get_primitives()
    atm = ref[0] == w.params["rho_atm"]
    assert atm.sum() > 1000 and np.array_equal(got[0] == w.params["rho_atm"], atm)
    assert np.all(got[1:4][:, atm] == 0) and np.all(got[4][atm] == w.params["p_atm"])
    assert_parity(got, ref, TOL64_SUB, "tov floors")
    hz.close()


def test_errors_and_call_order():
    from paper_1102_5202_b200 import Horizon, HzError
    from paper_1102_5202_b200.binding import HZ_EINVAL, HZ_ESTATE
    n = (8, 8, 8)
    a, b, g = wl.minkowski(n)
    p = np.zeros((8, 8, 8, 8))
    p[0], p[4] = 1.0, 1.0
    hz = Horizon(n, (1, 1, 1), (1, 1, 1))
    with pytest.raises(HzError) as e:
        hz.set_primitives(p)           # before the metric
    assert e.value.code == HZ_ESTATE
    with pytest.raises(HzError) as e:
        hz.step(0.1, 1)
    assert e.value.code == HZ_ESTATE
    bad = g.copy(); bad[0, 3, 3, 3] = -1.0
    with pytest.raises(HzError) as e:
        hz.set_metric(a, b, bad)       # not positive definite
    assert e.value.code == HZ_EINVAL
    bad_a = a.copy(); bad_a[1, 1, 1] = np.nan
    with pytest.raises(HzError):
        hz.set_metric(bad_a, b, g)
    hz.set_metric(a, b, g)
    for f, val in ((0, 0.0), (0, -1.0), (4, -1e-3), (1, 1.0), (5, np.inf), (2, np.nan)):
        q = p.copy(); q[f, 2, 3, 4] = val
        with pytest.raises(HzError) as e:
            hz.set_primitives(q)
        assert e.value.code == HZ_EINVAL, (f, val)
        with pytest.raises(HzError):
            hz.step(0.1, 1)            # still no valid primitives
    hz.set_primitives(p)
    with pytest.raises(HzError):
        hz.step(-0.1, 1)
    hz.substeps(0.1, 1)
    with pytest.raises(HzError) as e:
        hz.step(0.1, 1)                # in the middle of a step
    assert e.value.code == HZ_ESTATE
    hz.substeps(0.1, 2)
    hz.step(0.1, 1)
    assert np.abs(hz.get_primitives() - p).max() < 1e-14
    with pytest.raises(ValueError):
        hz.set_primitives(p[:, :4])
    hz.close()


@pytest.mark.parametrize("make,parts,dtype", [
    (lambda: wl.alfven_wave(n=(19, 12, 20)), 2, "f64"),     # periodic in z: the wrap-around is a neighbour
    (lambda: wl.alfven_wave(n=(19, 12, 21)), 3, "f64"),     # uneven slabs
    (lambda: wl.kerr_sweep(24), 3, "f64"),                  # outflow ends, curved metric (metric halos matter)
    (lambda: wl.kerr_sweep(24), 2, "f32"),
    (lambda: wl.blast(20), 4, "f32h"),
])
def test_slab_decomposition_reproduces_the_single_domain_bitwise(make, parts, dtype):
    """Row f3: the domain cut into slabs along z, ghost planes exchanged through
    hz_halo_pack / hz_halo_unpack after every substep, must give the single-context result bit for bit
    (same per-face and per-cell arithmetic; only where the ghost values come from differs)."""
    from paper_1102_5202_b200 import SlabGroup
    w = make()
    one = horizon(w, dtype)
    grp = SlabGroup(w, parts, dtype)
    one.substeps(w.dt, 4)
    grp.substeps(w.dt, 4)
    a, b = one.get_primitives(), grp.get_primitives()
    assert a.shape == b.shape
    assert np.array_equal(a, b), f"max |diff| = {np.abs(a - b).max()}"
    da, db = one.diagnostics(), grp.diagnostics()
    for k in ("c2p_fail", "atm_reset", "p_floor"):
        assert da[k] == db[k]
    for k in ("divB_max", "max_speed_over_dx"):
        assert da[k] == db[k]
    for k in ("sumD", "sumTau", "sumBx", "divB_L1"):
        assert abs(da[k] - db[k]) <= 1e-12 * max(abs(da[k]), 1e-300) + 1e-30, k
    one.close()
    grp.close()


@pytest.mark.parametrize("make,parts,dtype", [
    (lambda: wl.alfven_wave(n=(19, 12, 20)), 2, "f64"),     # periodic ring of two: both neighbours are the same slab
    (lambda: wl.alfven_wave(n=(19, 12, 21)), 3, "f64"),     # uneven slabs, periodic in x and y: ghost images travel too
    (lambda: wl.kerr_sweep(24), 3, "f64"),                  # outflow ends, curved metric
    (lambda: wl.kerr_sweep(24), 2, "f32"),
    (lambda: wl.blast(20), 4, "f32h"),
    (lambda: dataclasses.replace(wl.alfven_wave(n=(19, 12, 21)),
                                 params={**wl.alfven_wave(n=(19, 12, 21)).params, "recon": 1}), 3, "f64"),   # PPM: 3 planes
])
def test_exchange_fused_into_the_substep_reproduces_the_single_domain_bitwise(make, parts, dtype):
    """Row f3 / SURVEY 8(e): with the neighbours' primitive buffers attached (hz_peer_attach) the substep kernel
    stores the planes next to a cut straight into the neighbour's ghost planes -- no pack / unpack launches between
    substeps -- and the result is the single-context one bit for bit, like the pack / unpack path's."""
    from paper_1102_5202_b200 import SlabGroup
    w = make()
    one = horizon(w, dtype)
    grp = SlabGroup(w, parts, dtype, fused=True)
    n0 = sum(s.hz.launch_count() for s in grp.slabs)
    one.substeps(w.dt, 5)
    grp.substeps(w.dt, 5)
    assert sum(s.hz.launch_count() for s in grp.slabs) - n0 == 5 * parts     # nothing but the substep kernels
    a, b = one.get_primitives(), grp.get_primitives()
    assert np.array_equal(a, b), f"max |diff| = {np.abs(a - b).max()}"
    da, db = one.diagnostics(), grp.diagnostics()
    for k in ("c2p_fail", "atm_reset", "p_floor", "divB_max", "max_speed_over_dx"):
        assert da[k] == db[k]
    one.close()
    grp.close()


def test_peer_attach_reports_errors_and_detach_returns_to_pack_unpack():
    from paper_1102_5202_b200 import SlabGroup
    from paper_1102_5202_b200 import binding as B
    w = wl.kerr_sweep(24)
    one = horizon(w, "f64")
    p0, p1, fs = one.prim_buffers()
    assert p0 and p1 and p0 != p1 and fs > 24 ** 3
    with pytest.raises(B.HzError):            # no external side on a whole domain
        one.peer_attach(0, p0, p1, fs, 24)
    grp = SlabGroup(w, 3, "f64", fused=True)
    lo = grp.slabs[0]
    with pytest.raises(B.HzError):            # the low side of the lowest slab is the domain's outflow end
        lo.hz.peer_attach(0, p0, p1, fs, 8)
    with pytest.raises(B.HzError):            # side out of range
        lo.hz.peer_attach(2, p0, p1, fs, 8)
    # the general-mode kernels have no peer stores
    wg = dataclasses.replace(w, params={**w.params, "energy_var": 1})
    gg = SlabGroup(wg, 2, "f64")
    q0, q1, qfs = gg.slabs[1].hz.prim_buffers()
    with pytest.raises(B.HzError):
        gg.slabs[0].hz.peer_attach(1, q0, q1, qfs, gg.slabs[1].nz)
    gg.close()
    # detached, a slab is back under the rule of hz_halo_unpack: stepping twice without an exchange is refused
    one.substeps(w.dt, 2)
    grp.substeps(w.dt, 1)
    for s in grp.slabs:
        for side in (0, 1):
            s.hz.peer_detach(side)
    grp.fused = False
    grp.substeps(w.dt, 1)
    assert np.array_equal(one.get_primitives(), grp.get_primitives())
    grp.slabs[1].hz.substeps(w.dt, 1)
    with pytest.raises(B.HzError):
        grp.slabs[1].hz.substeps(w.dt, 1)
    one.close()
    grp.close()


def test_halo_calls_report_errors():
    from paper_1102_5202_b200 import binding as B
    import torch
    w = wl.shock_tube(64, axis=0)            # z inactive
    hz = horizon(w, "f64")
    with pytest.raises(B.HzError) as e:
        hz.halo_bytes(B.HZ_HALO_PRIM)
    assert e.value.code == B.HZ_EINVAL
    hz.close()
    w = wl.alfven_wave(n=(8, 8, 8))
    hz = horizon(w, "f64")
    nbytes = hz.halo_bytes(B.HZ_HALO_PRIM)
    assert nbytes == 9 * 2 * hz.halo_bytes(B.HZ_HALO_METRIC) // (10 * 2)
    host = np.empty(nbytes, dtype=np.uint8)
    with pytest.raises(B.HzError) as e:
        hz.halo_pack(B.HZ_HALO_PRIM, 0, host)          # host memory is refused
    assert e.value.code == B.HZ_EINVAL
    buf = torch.empty(nbytes, dtype=torch.uint8, device="cuda")
    with pytest.raises(B.HzError) as e:
        hz.halo_pack(B.HZ_HALO_PRIM, 2, buf)
    assert e.value.code == B.HZ_EINVAL
    hz.halo_pack(B.HZ_HALO_PRIM, 1, buf)
    hz.halo_unpack(B.HZ_HALO_PRIM, 1, buf)
    hz.close()


def test_external_slab_refuses_to_step_on_stale_ghost_planes():
    """a slab with an external z side whose ghost planes were never supplied (or not refreshed
    after a substep or after hz_set_primitives) used to stream zeros or stale planes and return HZ_OK.  Now
    hz_substeps / hz_step return HZ_ESTATE until both the metric's and the primitives' planes are in place."""
    import torch
    from paper_1102_5202_b200 import binding as B
    from paper_1102_5202_b200.slab import Slab
    w = wl.kerr_sweep(16)
    s = Slab(w, 0, 2, "f64")                      # low half: outflow below, EXTERNAL above
    s.set_metric()
    s.set_primitives()
    with pytest.raises(B.HzError) as e:
        s.hz.substeps(w.dt, 1)                    # no ghost planes at all
    assert e.value.code == B.HZ_ESTATE
    mbuf = torch.empty(s.hz.halo_bytes(B.HZ_HALO_METRIC), dtype=torch.uint8, device="cuda")
    pbuf = torch.empty(s.hz.halo_bytes(B.HZ_HALO_PRIM), dtype=torch.uint8, device="cuda")
    s.hz.halo_pack(B.HZ_HALO_METRIC, 1, mbuf)     # (any finite planes will do for this test: its own)
    s.hz.halo_unpack(B.HZ_HALO_METRIC, 1, mbuf)
    with pytest.raises(B.HzError) as e:
        s.hz.substeps(w.dt, 1)                    # metric planes supplied, primitives still missing
    assert e.value.code == B.HZ_ESTATE
    s.hz.halo_pack(B.HZ_HALO_PRIM, 1, pbuf)
    s.hz.halo_unpack(B.HZ_HALO_PRIM, 1, pbuf)
    s.hz.substeps(w.dt, 1)                        # complete: one substep goes through
    assert np.isfinite(s.hz.get_primitives()).all()
    with pytest.raises(B.HzError) as e:
        s.hz.substeps(w.dt, 1)                    # ... and outdates the primitives' planes again
    assert e.value.code == B.HZ_ESTATE
    with pytest.raises(B.HzError):
        s.hz.step(w.dt, 1)
    s.hz.halo_pack(B.HZ_HALO_PRIM, 1, pbuf)
    s.hz.halo_unpack(B.HZ_HALO_PRIM, 1, pbuf)
    s.hz.substeps(w.dt, 1)
    s.set_primitives()                            # new primitives: their planes are outdated too
    with pytest.raises(B.HzError) as e:
        s.hz.substeps(w.dt, 1)
    assert e.value.code == B.HZ_ESTATE
    s.hz.close()


def test_weak_scaling_slabs_generated_rank_by_rank_reproduce_the_single_box_bitwise():
    """bench.py --shard-weak (the paper's 120^3 -> 240 x 120^2 shape): every rank generates only its
    own n^3 slab of the n x n x (n N) Kerr-Schild box.  Three such slabs on one GPU, fed with the rank-by-rank
    inputs, must give bit for bit what a single context gives on the same inputs put together."""
    import dataclasses as dc
    from paper_1102_5202_b200 import SlabGroup
    n, parts = 14, 3
    slabs = [wl.kerr_sweep(n, zmult=parts, zslab=(r * n, (r + 1) * n)) for r in range(parts)]
    g = max(s.extra["bn_max"] for s in slabs)
    for s in slabs:
        s.prim8[5:8] *= s.extra["bn_max"] / g
    cat = lambda f: np.ascontiguousarray(np.concatenate([getattr(s, f) for s in slabs], axis=-3))
    whole = dc.replace(slabs[0], n=(n, n, n * parts), alpha=cat("alpha"), beta3=cat("beta3"), gamma6=cat("gamma6"),
                       prim8=cat("prim8"))
    one = horizon(whole, "f64")
    grp = SlabGroup(slabs, parts, "f64")
    one.substeps(whole.dt, 4)
    grp.substeps(whole.dt, 4)
    assert np.array_equal(one.get_primitives(), grp.get_primitives())
    one.close()
    grp.close()


def _paper_sp_dp():
    import os
    out = {}
    with open(os.path.join(os.path.dirname(__file__), "golden", "paper_sp_minus_dp.txt")) as f:
        for line in f:
            if line.strip() and not line.startswith("#"):
                k, v = line.split()[:2]
                out[k] = float(v)
    return out


def test_fp32_minus_fp64_after_the_full_tube_run_is_of_the_papers_order():
    """PAPER.md:286-298 compares its single- and double-precision runs of the shock tubes: differences of
    5e-5 (rho) and 1e-4 (u^x) at the shock, < 1e-6 in smooth flow.  Config 1 to t = 0.4 here: the largest
    fp32 - fp64 difference of any primitive must stay within the paper's at-the-shock figure, and the
    smooth left state (x < -0.45, untouched by any wave) within its smooth-flow figure."""
    ref = _paper_sp_dp()
    w = wl.shock_tube(400)
    res = {}
    for dt in ("f64", "f32"):
        hz = horizon(w, dt)
        hz.step(w.dt, w.nsteps)
        res[dt] = hz.get_primitives().astype(np.float64)
        assert hz.diagnostics()["c2p_fail"] == 0
        hz.close()
    d = np.abs(res["f32"] - res["f64"])
    assert d.max() <= ref["sod_shock_ux"], d.reshape(8, -1).max(axis=1)
    assert d[..., :20].max() <= ref["sod_smooth"], d[..., :20].max()


def test_pure_fp32_recovery_does_not_fail_in_the_magnetised_blast():
    """In the blast's ambient medium B^2 > rho h, so the Newton step of the fp32 recovery cannot fall below
    eps (Z + B^2): the convergence test is made against that scale (hz_physics.cuh).  Without it 256 cells
    of this run were reset to atmosphere and v differed from fp64 by 1e-2; with it, by ~1e-6."""
    w = wl.blast(64)
    res = {}
    for dt in ("f64", "f32"):
        hz = horizon(w, dt)
        hz.step(w.dt, 20)
        res[dt] = hz.get_primitives().astype(np.float64)
        d = hz.diagnostics()
        assert d["c2p_fail"] == 0 and d["atm_reset"] == 0, d
        hz.close()
    diff = np.abs(res["f32"] - res["f64"])
    assert diff[1:4].max() <= 1e-4 and diff[0].max() <= 1e-6 and diff[4].max() <= 1e-4, diff.reshape(8, -1).max(axis=1)


@pytest.mark.parametrize("name", ["tube_x", "alfven_3d", "blast", "tov", "kerr"])
def test_two_unknown_recovery_scheme_parity_and_agreement(name):
    """Row f4 (the second con2prim scheme): Newton on (Z, v^2).  GPU against the oracle running
    the same scheme at the fp64 bar after a full RK3 step; and, the root being unique, against the GPU's
    own one-unknown run far below that bar.  fp32 at its bar."""
    w = SMALL[name]()
    w2 = dataclasses.replace(w, params={**w.params, "c2p_scheme": 1})
    o = oracle_for(w2)
    o.substeps(w.dt, 3)
    ref = o.get_primitives()
    hz2 = horizon(w2, "f64")
    hz2.substeps(w.dt, 3)
    got2 = hz2.get_primitives()
    assert_parity(got2, ref, TOL64_SUB, f"{name} two-unknown scheme")
    d2 = hz2.diagnostics()
    do = o.diagnostics()
    for k in ("c2p_fail", "atm_reset", "p_floor"):
        assert d2[k] == do[k], (k, d2[k], do[k])
    hz1 = horizon(w, "f64")
    hz1.substeps(w.dt, 3)
    assert_parity(got2, hz1.get_primitives(), 1e-11, f"{name} two-unknown vs one-unknown")
    hz1.close()
    hz2.close()
    hz32 = horizon(w2, "f32")
    o1 = oracle_for(w2)
    o1.substeps(w.dt, 1)
    hz32.substeps(w.dt, 1)
    got = hz32.get_primitives()
    ref1 = o1.get_primitives()
    flips = floor_flip_mask(got, ref1, w.params["rho_atm"], w.params["atm_tol"])
    assert flips.sum() <= 2e-4 * w.ncell
    assert_parity(got, ref1, TOL32_SUB, f"{name} two-unknown scheme fp32", mask=flips)
    hz32.close()


@pytest.mark.parametrize("name", ["tube_x", "alfven_3d", "tov", "kerr"])
def test_papers_energy_variable_parity(name):
    """Row f4 / reading R1b: evolve the paper's -sqrt(-g) T^t_t instead of sqrt(gamma) tau.
    GPU against the oracle running the same option: primitives and the conserved set (slot 4 carries the
    paper's variable) at the fp64 bar after a full RK3 step."""
    w = SMALL[name]()
    w1 = dataclasses.replace(w, params={**w.params, "energy_var": 1})
    o = oracle_for(w1)
    hz = horizon(w1, "f64")
    o.substeps(w.dt, 3)
    hz.substeps(w.dt, 3)
    assert_parity(hz.get_primitives(), o.get_primitives(), TOL64_SUB, f"{name} energy variable")
    Uo, Ug = o.get_conserved(), hz.get_conserved()
    den = np.abs(Uo[4]).sum()
    assert np.abs(Ug[4] - Uo[4]).sum() <= TOL64_SUB * den
    do, dg = o.diagnostics(), hz.diagnostics()
    for k in ("c2p_fail", "atm_reset", "p_floor"):
        assert do[k] == dg[k]
    hz.close()


def test_papers_energy_variable_is_conserved_to_roundoff_on_the_gpu():
    """no energy source on a time-independent metric.  Periodic box, smooth space-dependent
    lapse, shift and 3-metric: the sum of the paper's variable stays put to round-off over 30 substeps in
    fp64, while sum(sqrt(gamma) tau) of the default form moves (its source is at work)."""
    from test_oracle_grid import _wavy_metric_workload
    w = _wavy_metric_workload(40)
    w1 = dataclasses.replace(w, params={**w.params, "energy_var": 1})
    a, b = horizon(w, "f64"), horizon(w1, "f64")
    t0, e0 = a.diagnostics()["sumTau"], b.diagnostics()["sumTau"]
    a.step(w.dt, 10)
    b.step(w.dt, 10)
    t1, e1 = a.diagnostics()["sumTau"], b.diagnostics()["sumTau"]
    assert abs(e1 - e0) <= 1e-13 * abs(e0), (e0, e1)
    assert abs(t1 - t0) >= 1e-7 * abs(t0), (t0, t1)
    a.close()
    b.close()


@pytest.mark.parametrize("name", ["tube_x_ragged", "tube_z", "alfven_3d", "alfven_2d", "blast", "tov", "kerr"])
def test_ppm_reconstruction_parity(name):
    """Row f1: PPM instead of the MC-limited linear reconstruction -- 3 ghost layers, its own
    tiles.  GPU against the oracle running PPM: fp64 at 1e-10 after 1 and 3 substeps, fp32 and the mixed mode
    at 1e-4 after one substep."""
    w = SMALL[name]()
    wp = dataclasses.replace(w, params={**w.params, "recon": 1})
    o = oracle_for(wp)
    hz = horizon(wp, "f64")
    o.substeps(w.dt, 1)
    hz.substeps(w.dt, 1)
    ref1 = o.get_primitives()
    assert_parity(hz.get_primitives(), ref1, TOL64_SUB, f"{name} PPM 1 substep")
    o.substeps(w.dt, 2)
    hz.substeps(w.dt, 2)
    assert_parity(hz.get_primitives(), o.get_primitives(), TOL64_SUB, f"{name} PPM 3 substeps")
    do, dg = o.diagnostics(), hz.diagnostics()
    for k in ("c2p_fail", "atm_reset", "p_floor"):
        assert do[k] == dg[k], (k, do[k], dg[k])
    hz.close()
    for dt in ("f32", "f32h"):
        h32 = horizon(wp, dt)
        h32.substeps(w.dt, 1)
        got = h32.get_primitives()
        flips = floor_flip_mask(got, ref1, w.params["rho_atm"], w.params["atm_tol"])
        assert flips.sum() <= 2e-4 * w.ncell
        assert_parity(got, ref1, TOL32_SUB, f"{name} PPM {dt}", mask=flips)
        h32.close()


def test_ppm_differs_from_mc_and_slabs_exchange_three_planes():
    """PPM is not MC in disguise (the two runs differ at truncation level), and the slab decomposition with
    its 3-plane halo reproduces the single domain bitwise."""
    from paper_1102_5202_b200 import SlabGroup
    w = wl.alfven_wave(n=(19, 12, 21))
    wp = dataclasses.replace(w, params={**w.params, "recon": 1})
    a, b = horizon(w, "f64"), horizon(wp, "f64")
    a.substeps(w.dt, 3)
    b.substeps(w.dt, 3)
    pa, pb = a.get_primitives(), b.get_primitives()
    assert np.abs(pa - pb).max() > 1e-6
    grp = SlabGroup(wp, 3, "f64")
    grp.substeps(w.dt, 3)
    assert np.array_equal(grp.get_primitives(), pb)
    assert grp.slabs[0].hz.halo_bytes(0) == 9 * 3 * (grp.slabs[0].hz.halo_bytes(1) // (10 * 3))
    a.close(); b.close(); grp.close()


@pytest.mark.parametrize("name", ["kerr", "tov", "alfven_3d"])
def test_all_options_together_parity(name):
    """PPM + the two-unknown recovery + the paper's energy variable in one run (the options are independent
    switches in hz_params; this guards their combination), fp64 bar after a full RK3 step, and the mixed mode
    at the fp32 bar after one substep."""
    w = SMALL[name]()
    wo = dataclasses.replace(w, params={**w.params, "recon": 1, "c2p_scheme": 1, "energy_var": 1})
    o = oracle_for(wo)
    hz = horizon(wo, "f64")
    o.substeps(w.dt, 1)
    ref1 = o.get_primitives()
    o.substeps(w.dt, 2)
    hz.substeps(w.dt, 3)
    assert_parity(hz.get_primitives(), o.get_primitives(), TOL64_SUB, f"{name} all options")
    Uo, Ug = o.get_conserved(), hz.get_conserved()
    assert np.abs(Ug[4] - Uo[4]).sum() <= TOL64_SUB * np.abs(Uo[4]).sum()
    hz.close()
    hm = horizon(wo, "f32h")
    hm.substeps(w.dt, 1)
    got = hm.get_primitives()
    flips = floor_flip_mask(got, ref1, w.params["rho_atm"], w.params["atm_tol"])
    assert flips.sum() <= 2e-4 * w.ncell
    assert_parity(got, ref1, TOL32_SUB, f"{name} all options mixed", mask=flips)
    hm.close()


def test_fma_peak_is_plausible():
    """hz_fma_peak: the measured FMA-pipe throughput the ALU roofline is compared with.  fp32 issues at twice
    the fp64 rate on this part; both must be positive and below the derived unit-count peak."""
    from paper_1102_5202_b200.binding import fma_peak
    f64, f32 = fma_peak("f64"), fma_peak("f32")
    assert 1.0 < f64 < 148 * 64 * 2 * 2.1e9 / 1e12 * 1.02
    assert 1.0 < f32 < 148 * 128 * 2 * 2.1e9 / 1e12 * 1.02
    assert 1.5 < f32 / f64 < 2.5
