"""Seeded synthetic input generators for the five BASELINE.json configs.

This module serves BOTH the CPU oracle (tests) and the CUDA path (tests, bench.py).  It holds none of
the method's arithmetic: it only produces the API inputs -- lapse, shift, 3-metric and the eight API
primitives (rho, v^i, p, B^i) on cell centres -- plus grid, boundary and parameter choices.  Everything
is float64 numpy, shape (planes, nz, ny, nx), x fastest.  It imports neither `oracle` nor
`paper_1102_5202_b200`.

The paper's own workloads (RNS stellar models) are not available; these inputs stand
in for them with the same shapes: a magnetised tube, a star on a fixed metric
(PAPER.md:206-210), cubic grids.
"""
from dataclasses import dataclass, field

import numpy as np

BC_PERIODIC, BC_OUTFLOW = 0, 1


@dataclass
class Workload:
    name: str
    n: tuple            # (nx, ny, nz)
    h: tuple            # (dx, dy, dz)
    bc: tuple           # per axis
    params: dict        # gamma_ad, rho_atm, p_atm, atm_tol, cleaning, kappa
    alpha: np.ndarray   # (nz, ny, nx)
    beta3: np.ndarray   # (3, nz, ny, nx)
    gamma6: np.ndarray  # (6, nz, ny, nx)  xx, xy, xz, yy, yz, zz
    prim8: np.ndarray   # (8, nz, ny, nx)  rho, vx, vy, vz, p, Bx, By, Bz
    dt: float
    nsteps: int         # full RK3 steps of the BASELINE run
    extra: dict = field(default_factory=dict)

    @property
    def ncell(self):
        return self.n[0] * self.n[1] * self.n[2]


def centres(n, lo, hi):
    """Cell-centre coordinates of n cells on [lo, hi]."""
    h = (hi - lo) / n
    return lo + (np.arange(n) + 0.5) * h, h


def minkowski(n):
    nx, ny, nz = n
    alpha = np.ones((nz, ny, nx))
    beta3 = np.zeros((3, nz, ny, nx))
    gamma6 = np.zeros((6, nz, ny, nx))
    gamma6[0] = gamma6[3] = gamma6[5] = 1.0
    return alpha, beta3, gamma6


def constant_metric(n, alpha=0.8, beta=(0.1, -0.2, 0.05),
                    gamma=(1.3, 0.2, -0.1, 0.9, 0.15, 1.1)):
    """Constant but non-trivial metric (pin P3): non-diagonal SPD gamma_ij, non-zero shift."""
    nx, ny, nz = n
    a = np.full((nz, ny, nx), float(alpha))
    b = np.empty((3, nz, ny, nx))
    g = np.empty((6, nz, ny, nx))
    for i in range(3):
        b[i] = beta[i]
    for i in range(6):
        g[i] = gamma[i]
    return a, b, g


# -------------------------------------------------------------------------------------------------
# Config 1: magnetised shock tube ("Balsara 1"; BASELINE.json config 1 binds the values)
# -------------------------------------------------------------------------------------------------
def shock_tube(nx=400, axis=0, mirror=False, t_end=0.4, cfl=0.4):
    n = [1, 1, 1]
    n[axis] = nx
    x, dx = centres(nx, -0.5, 0.5)
    left = x < 0
    if mirror:
        left = x > 0
    shp = [1, 1, 1]
    shp[2 - axis] = nx
    L = left.reshape(shp)
    nzyx = (n[2], n[1], n[0])
    prim = np.zeros((8,) + nzyx)
    prim[0] = np.where(L, 1.0, 0.125)
    prim[4] = np.where(L, 1.0, 0.1)
    t1 = (axis + 1) % 3
    prim[5 + axis] = 0.5
    prim[5 + t1] = np.where(L, 1.0, -1.0)
    alpha, beta3, gamma6 = minkowski(n)
    h = [1.0, 1.0, 1.0]
    h[axis] = dx
    bc = [BC_PERIODIC] * 3
    bc[axis] = BC_OUTFLOW
    dt = cfl * dx
    params = dict(gamma_ad=2.0, rho_atm=1e-12, p_atm=1e-14, atm_tol=1e-3, cleaning=1, kappa=1.0)
    return Workload("tube", tuple(n), tuple(h), tuple(bc), params, alpha, beta3, gamma6, prim, dt,
                    int(round(t_end / dt)), dict(x=x))


# -------------------------------------------------------------------------------------------------
# Config 2: circularly polarised Alfven wave along the cube diagonal
# -------------------------------------------------------------------------------------------------
ALFVEN_VA = (3.0 - np.sqrt(5.0)) / 2.0  # closed form for rho=p=B0=eta=1, Gamma=4/3 (P8)


def alfven_fields(n, t=0.0, direction="diag"):
    """Exact solution at time t on the periodic unit cube (the initial data at t = 0)."""
    nx, ny, nz = n
    x, dx = centres(nx, 0.0, 1.0)
    y, dy = centres(ny, 0.0, 1.0)
    z, dz = centres(nz, 0.0, 1.0)
    Z, Y, X = np.meshgrid(z, y, x, indexing="ij")
    if direction == "diag":
        nh = np.array([1.0, 1.0, 1.0]) / np.sqrt(3.0)
        e1 = np.array([1.0, -1.0, 0.0]) / np.sqrt(2.0)
        e2 = np.array([1.0, 1.0, -2.0]) / np.sqrt(6.0)
        kmag = 2 * np.pi * np.sqrt(3.0)
        s = (X + Y + Z) / np.sqrt(3.0)
    elif direction == "x":
        nh, e1, e2 = np.eye(3)
        kmag = 2 * np.pi
        s = X + 0 * Y + 0 * Z
    else:
        raise ValueError(direction)
    B0, eta, vA = 1.0, 1.0, ALFVEN_VA
    phi = kmag * (s - vA * t)
    c, sn = np.cos(phi), np.sin(phi)
    prim = np.zeros((8, nz, ny, nx))
    prim[0] = 1.0
    prim[4] = 1.0
    for i in range(3):
        prim[1 + i] = -vA * eta * (c * e1[i] + sn * e2[i])
        prim[5 + i] = B0 * nh[i] + eta * B0 * (c * e1[i] + sn * e2[i])
    period = 2 * np.pi / (kmag * vA)
    return prim, (dx, dy, dz), period


def alfven_wave(nx=64, direction="diag", cfl=0.25, n=None):
    if n is None:
        n = (nx, nx, nx) if direction == "diag" else (nx, 1, 1)
    prim, h, period = alfven_fields(n, 0.0, direction)
    alpha, beta3, gamma6 = minkowski(n)
    hmin = min(hh for hh, nn in zip(h, n) if nn > 1)
    nsteps = int(np.ceil(period / (cfl * hmin)))
    dt = period / nsteps  # lands exactly on one period
    params = dict(gamma_ad=4.0 / 3.0, rho_atm=1e-12, p_atm=1e-14, atm_tol=1e-3, cleaning=1, kappa=1.0)
    return Workload("alfven", tuple(n), tuple(h), (BC_PERIODIC,) * 3, params, alpha, beta3, gamma6, prim, dt,
                    nsteps, dict(period=period, direction=direction))


# -------------------------------------------------------------------------------------------------
# Config 3: cylindrical magnetised blast wave
# -------------------------------------------------------------------------------------------------
def blast(nx=128, cfl=0.25, nsteps=67):
    n = (nx, nx, nx)
    x, dx = centres(nx, -6.0, 6.0)
    Z, Y, X = np.meshgrid(x, x, x, indexing="ij")
    r = np.sqrt(X * X + Y * Y)
    w = np.clip((1.0 - r) / (1.0 - 0.8), 0.0, 1.0)  # 1 inside r<0.8, 0 outside r>1, linear between
    prim = np.zeros((8,) + Z.shape)
    prim[0] = 1e-4 + (1e-2 - 1e-4) * w
    prim[4] = 5e-4 + (1.0 - 5e-4) * w
    prim[5] = 0.1
    alpha, beta3, gamma6 = minkowski(n)
    params = dict(gamma_ad=4.0 / 3.0, rho_atm=1e-7, p_atm=1e-9, atm_tol=1e-3, cleaning=1, kappa=1.0)
    return Workload("blast", n, (dx, dx, dx), (BC_OUTFLOW,) * 3, params, alpha, beta3, gamma6, prim, cfl * dx,
                    nsteps)


# -------------------------------------------------------------------------------------------------
# Config 4: magnetised TOV star on a fixed spacetime
# -------------------------------------------------------------------------------------------------
def tov_solve(K=100.0, Gamma=2.0, rho_c=1.28e-3, rtol=1e-12):
    """TOV in areal radius r, with the isotropic radius integrated alongside.  G = c = Msun = 1."""
    from scipy.integrate import solve_ivp

    def eos_rho(p):
        return (max(p, 0.0) / K) ** (1.0 / Gamma)

    def rhs(r, y):
        m, p, nu, lnq = y  # q = r_iso / r
        rho = eos_rho(p)
        e = rho + p / (Gamma - 1.0)
        if r < 1e-12:
            return [0.0, 0.0, 0.0, 0.0]
        f = 1.0 - 2.0 * m / r
        dnu = (m + 4 * np.pi * r ** 3 * p) / (r * r * f)
        return [4 * np.pi * r * r * e, -(e + p) * dnu, dnu, (1.0 / np.sqrt(f) - 1.0) / r]

    p_c = K * rho_c ** Gamma
    e_c = rho_c + p_c / (Gamma - 1.0)
    r0 = 1e-6
    y0 = [4 * np.pi / 3 * e_c * r0 ** 3, p_c - 2 * np.pi / 3 * (e_c + p_c) * (e_c + 3 * p_c) * r0 ** 2, 0.0, 0.0]

    def surface(r, y):
        return y[1] - 1e-14 * p_c

    surface.terminal = True
    surface.direction = -1
    sol = solve_ivp(rhs, [r0, 50.0], y0, method="DOP853", rtol=rtol, atol=[1e-15, 1e-21, 1e-15, 1e-15],
                    events=surface, max_step=0.02)
    R = sol.t[-1]
    M = sol.y[0, -1]
    # match lapse and isotropic radius to the exterior Schwarzschild solution
    nu_shift = 0.5 * np.log(1.0 - 2.0 * M / R) - sol.y[2, -1]
    Riso = 0.5 * (np.sqrt(R * R - 2 * M * R) + R - M)
    lnq_shift = np.log(Riso / R) - sol.y[3, -1]
    r = sol.t
    m, p, nu, lnq = sol.y
    riso = r * np.exp(lnq + lnq_shift)
    return dict(r=r, riso=riso, m=m, p=np.maximum(p, 0.0), alpha=np.exp(nu + nu_shift), M=M, R=R, Riso=Riso,
                K=K, Gamma=Gamma, rho_c=rho_c, p_c=p_c, alpha_c=float(np.exp(sol.y[2, 0] + nu_shift)),
                alpha_s=float(np.sqrt(1 - 2 * M / R)))


def _tov_profiles(tov, riso_q):
    """Sample alpha, psi^4, rho, p at isotropic radii riso_q (any shape) by cubic interpolation."""
    from scipy.interpolate import CubicSpline

    rs, M = tov["riso"], tov["M"]
    inside = riso_q < tov["Riso"]
    rq = np.clip(riso_q, rs[0], rs[-1])
    sp_r = CubicSpline(rs, tov["r"])
    sp_a = CubicSpline(rs, tov["alpha"])
    sp_p = CubicSpline(rs, tov["p"])
    r_areal = sp_r(rq)
    psi4_in = (r_areal / rq) ** 2
    x = M / (2.0 * np.maximum(riso_q, rs[0]))
    psi4 = np.where(inside, psi4_in, (1.0 + x) ** 4)
    alpha = np.where(inside, sp_a(rq), (1.0 - x) / (1.0 + x))
    p = np.where(inside, np.maximum(sp_p(rq), 0.0), 0.0)
    rho = (p / tov["K"]) ** (1.0 / tov["Gamma"])
    return alpha, psi4, rho, p


def _curl_field(Ahat_ext, X, Y, sqrtg, h):
    """B^i = eps^{ijk} d_j A_k / sqrt(gamma) with A = (-y Ahat, x Ahat, 0), centred differences (R19).

    Ahat_ext, X, Y are given on the grid extended by one layer on every side; sqrtg on the interior."""
    Ax = -Y * Ahat_ext
    Ay = X * Ahat_ext
    dx, dy, dz = h
    c = (slice(1, -1),) * 3

    def d(a, axis, hh):  # centred difference along array axis (0=z,1=y,2=x) on the interior
        sl_p, sl_m = [slice(1, -1)] * 3, [slice(1, -1)] * 3
        sl_p[axis], sl_m[axis] = slice(2, None), slice(0, -2)
        return (a[tuple(sl_p)] - a[tuple(sl_m)]) / (2 * hh)

    Bx = -d(Ay, 0, dz) / sqrtg
    By = d(Ax, 0, dz) / sqrtg
    Bz = (d(Ay, 2, dx) - d(Ax, 1, dy)) / sqrtg
    del c
    return Bx, By, Bz


def tov_star(nx=192, half_width=20.0, Omega=0.01, Bmax=1e-4, cfl=0.25, nsteps=167, tov=None,
             rho_atm=1e-10):
    tov = tov or tov_solve()
    n = (nx, nx, nx)
    x, dx = centres(nx, -half_width, half_width)
    xe = np.concatenate([[x[0] - dx], x, [x[-1] + dx]])  # one extra layer for the curl
    Ze, Ye, Xe = np.meshgrid(xe, xe, xe, indexing="ij")
    re = np.sqrt(Xe * Xe + Ye * Ye + Ze * Ze)
    alpha_e, psi4_e, rho_e, p_e = _tov_profiles(tov, re)
    c = (slice(1, -1),) * 3
    alpha, psi4, rho, p = alpha_e[c], psi4_e[c], rho_e[c], p_e[c]
    X, Y = Xe[c], Ye[c]
    K, Gam = tov["K"], tov["Gamma"]
    p_atm = K * rho_atm ** Gam
    star = rho > 10 * rho_atm
    prim = np.zeros((8,) + alpha.shape)
    prim[0] = np.where(rho > rho_atm, rho, rho_atm)
    prim[4] = np.where(rho > rho_atm, p, p_atm)
    prim[1] = np.where(star, -Omega * Y / alpha, 0.0)  # R20: coordinate angular velocity Omega, beta = 0
    prim[2] = np.where(star, Omega * X / alpha, 0.0)
    sqrtg = psi4 ** 1.5
    Ahat = np.maximum(p_e - 0.04 * tov["p_c"], 0.0) ** 2
    Bx, By, Bz = _curl_field(Ahat, Xe, Ye, sqrtg, (dx, dx, dx))
    Bnorm = np.sqrt(psi4 * (Bx * Bx + By * By + Bz * Bz))
    scale = Bmax / Bnorm.max() if Bnorm.max() > 0 else 0.0
    prim[5], prim[6], prim[7] = scale * Bx, scale * By, scale * Bz
    beta3 = np.zeros((3,) + alpha.shape)
    gamma6 = np.zeros((6,) + alpha.shape)
    gamma6[0] = gamma6[3] = gamma6[5] = psi4
    params = dict(gamma_ad=Gam, rho_atm=rho_atm, p_atm=p_atm, atm_tol=1e-3, cleaning=1, kappa=1.0)
    return Workload("tov", n, (dx, dx, dx), (BC_OUTFLOW,) * 3, params, np.ascontiguousarray(alpha), beta3, gamma6,
                    prim, cfl * dx, nsteps, dict(tov={k: v for k, v in tov.items() if np.isscalar(v)}))


# -------------------------------------------------------------------------------------------------
# Config 5: Kerr-Schild throughput sweep
# -------------------------------------------------------------------------------------------------
def kerr_schild(X, Y, Z, M=1.0, a=0.9):
    """Closed-form 3+1 Kerr-Schild: alpha, beta^i, gamma_ij (6) at Cartesian points (hole at origin)."""
    R2 = X * X + Y * Y + Z * Z
    r2 = 0.5 * ((R2 - a * a) + np.sqrt((R2 - a * a) ** 2 + 4 * a * a * Z * Z))
    r = np.sqrt(r2)
    H = M * r * r2 / (r2 * r2 + a * a * Z * Z)
    l = [(r * X + a * Y) / (r2 + a * a), (r * Y - a * X) / (r2 + a * a), Z / r]
    alpha = 1.0 / np.sqrt(1.0 + 2.0 * H)
    beta3 = np.stack([2.0 * H * li / (1.0 + 2.0 * H) for li in l])
    g = []
    for (i, j) in [(0, 0), (0, 1), (0, 2), (1, 1), (1, 2), (2, 2)]:
        g.append((1.0 if i == j else 0.0) + 2.0 * H * l[i] * l[j])
    return alpha, beta3, np.stack(g)


def gaussian_field(seed, x, y, z, side=12.0, nmodes=32, nmax=4):
    """Smooth unit-variance random field sum_m a_m cos(k_m.x + phi_m), k_m = 2 pi n_m / side (seeded)."""
    rng = np.random.default_rng(seed)
    nvec = rng.integers(-nmax, nmax + 1, size=(nmodes, 3))
    for m in range(nmodes):  # no zero mode
        while not nvec[m].any():
            nvec[m] = rng.integers(-nmax, nmax + 1, size=3)
    amp = rng.normal(size=nmodes) / np.sqrt(nmodes / 2.0)
    phase = rng.uniform(0, 2 * np.pi, size=nmodes)
    k = 2 * np.pi * nvec / side
    Ex = np.exp(1j * np.outer(k[:, 0], x))  # (m, nx)
    Ey = np.exp(1j * np.outer(k[:, 1], y))
    Ez = np.exp(1j * np.outer(k[:, 2], z)) * (amp * np.exp(1j * phase))[:, None]
    T = (Ey[:, :, None] * Ex[:, None, :]).reshape(nmodes, -1)  # (m, ny*nx)
    out = np.empty((len(z), len(y) * len(x)))
    for k0 in range(0, len(z), 16):  # blocked over z to bound the complex temporary
        out[k0:k0 + 16] = (Ez[:, k0:k0 + 16].T @ T).real
    return out.reshape(len(z), len(y), len(x))


def kerr_sweep(nx=128, cfl=0.25, nsteps=34, M=1.0, a=0.9, Bmax=1e-2, zmult=1, zslab=None):
    """BASELINE config 5.  zmult > 1 stacks zmult cubes along z -- the grid is nx x nx x (zmult nx) over
    z in [-6 zmult, 6 zmult] with the same spacing -- which is the shape of the paper's weak-scaling run
    (120^3 on one GPU against 240 x 120^2 on two).  zslab = (k0, k1) generates the z planes
    k0 .. k1-1 of that grid only (one rank's slab; no rank ever holds the whole box); the field is then scaled
    by the slab's own maximum, which extra['bn_max'] records so that the ranks can agree on the global one."""
    nz = nx * zmult
    k0, k1 = (0, nz) if zslab is None else zslab
    n = (nx, nx, k1 - k0)
    side = 12.0
    x, dx = centres(nx, 4.0, 16.0)
    y, _ = centres(nx, -6.0, 6.0)
    z = (-6.0 * zmult + (np.arange(k0, k1) + 0.5) * dx)
    ext = lambda c: np.concatenate([[c[0] - dx], c, [c[-1] + dx]])
    xe, ye, ze = ext(x), ext(y), ext(z)
    Ze, Ye, Xe = np.meshgrid(ze, ye, xe, indexing="ij")
    c = (slice(1, -1),) * 3
    alpha, beta3, gamma6 = kerr_schild(Xe[c], Ye[c], Ze[c], M, a)
    varpi_e = np.sqrt(Xe * Xe + Ye * Ye)
    G_e = gaussian_field(1102, xe, ye, ze, side)
    env_e = np.exp(-((varpi_e - 10.0) ** 2 + Ze * Ze) / 16.0)
    rho_e = 1e-2 * np.exp(0.5 * G_e) * env_e + 1e-6
    G5_e = gaussian_field(1105, xe, ye, ze, side)
    Ahat_e = np.maximum(rho_e - 2e-3, 0.0) * (1.0 + 0.3 * G5_e)
    del G_e, G5_e, env_e, varpi_e
    rho = rho_e[c]
    prim = np.zeros((8,) + rho.shape)
    prim[0] = rho
    prim[4] = 0.05 * rho
    w = np.stack([gaussian_field(s, x, y, z, side) for s in (5202, 5203, 5204)])
    w /= np.sqrt(1.0 + (w * w).sum(axis=0))  # Euclidean |w| < 1, grid independent
    gxx, gxy, gxz, gyy, gyz, gzz = gamma6
    wn = np.sqrt(gxx * w[0] ** 2 + gyy * w[1] ** 2 + gzz * w[2] ** 2 +
                 2 * (gxy * w[0] * w[1] + gxz * w[0] * w[2] + gyz * w[1] * w[2]))
    prim[1:4] = 0.5 * w / np.maximum(1.0, wn)
    det = (gxx * (gyy * gzz - gyz * gyz) - gxy * (gxy * gzz - gyz * gxz) + gxz * (gxy * gyz - gyy * gxz))
    sqrtg = np.sqrt(det)
    Bx, By, Bz = _curl_field(Ahat_e, Xe, Ye, sqrtg, (dx, dx, dx))
    Bn = np.sqrt(gxx * Bx * Bx + gyy * By * By + gzz * Bz * Bz + 2 * (gxy * Bx * By + gxz * Bx * Bz + gyz * By * Bz))
    scale = Bmax / Bn.max()
    prim[5], prim[6], prim[7] = scale * Bx, scale * By, scale * Bz
    params = dict(gamma_ad=4.0 / 3.0, rho_atm=1e-8, p_atm=1e-10, atm_tol=1e-3, cleaning=1, kappa=1.0)
    return Workload("kerr", n, (dx, dx, dx), (BC_OUTFLOW,) * 3, params, np.ascontiguousarray(alpha),
                    np.ascontiguousarray(beta3), np.ascontiguousarray(gamma6), prim, cfl * dx, nsteps,
                    dict(bn_max=float(Bn.max()), zmult=zmult, zslab=(k0, k1), nz_global=nz))


def random_states(seed, count, vmax=0.95, curved=True):
    """Random physical states + SPD metrics for point pins (P1, P2): prim8-like rows and met10 rows."""
    rng = np.random.default_rng(seed)
    met = np.zeros((count, 10))
    met[:, 0] = rng.uniform(0.5, 1.2, count)
    met[:, 1:4] = rng.uniform(-0.3, 0.3, (count, 3))
    if curved:
        A = rng.normal(size=(count, 3, 3)) * 0.25 + np.eye(3)
        g = np.einsum("nij,nkj->nik", A, A)
    else:
        met[:, 0] = 1.0
        met[:, 1:4] = 0.0
        g = np.broadcast_to(np.eye(3), (count, 3, 3)).copy()
    met[:, 4], met[:, 5], met[:, 6] = g[:, 0, 0], g[:, 0, 1], g[:, 0, 2]
    met[:, 7], met[:, 8], met[:, 9] = g[:, 1, 1], g[:, 1, 2], g[:, 2, 2]
    rho = 10 ** rng.uniform(-6, 0, count)
    p = rho * 10 ** rng.uniform(-4, 1, count)
    vdir = rng.normal(size=(count, 3))
    vn = np.sqrt(np.einsum("ni,nij,nj->n", vdir, g, vdir))
    v = vdir / vn[:, None] * rng.uniform(0, vmax, count)[:, None]
    W = 1 / np.sqrt(1 - np.einsum("ni,nij,nj->n", v, g, v))
    bdir = rng.normal(size=(count, 3))
    bn = np.sqrt(np.einsum("ni,nij,nj->n", bdir, g, bdir))
    B = bdir / bn[:, None] * np.sqrt(rho * 10 ** rng.uniform(-4, 2, count))[:, None]
    prim9 = np.zeros((count, 9))
    prim9[:, 0] = rho
    prim9[:, 1:4] = v * W[:, None]
    prim9[:, 4] = p
    prim9[:, 5:8] = B
    prim9[:, 8] = rng.normal(size=count) * 0.01
    return prim9, met
