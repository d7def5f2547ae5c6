"""Whole-RHS pins for the oracle (O4-O12): special cases that reduce to textbook schemes or to
analytic results, invariants, and the values the paper prints for its Couette case."""
import numpy as np
import pytest

import workloads as W
from oracle.fr_oracle import FROracle, common_flux, flux_inviscid

G = 1.4


def _coords(o):
    return np.asarray(o.xu_phys, dtype=np.float64)


def _state_on(o, fn, **kw):
    return np.ascontiguousarray(np.moveaxis(fn(_coords(o), **kw), -1, 1))


# ------------------------------------------------------------------------------------------
# p = 0 reduces to the first-order finite-volume scheme (SURVEY 8c "Whole RHS, special case")
# ------------------------------------------------------------------------------------------
def _fv_neighbours(nx, ny):
    """(element, direction, side) -> neighbour element on a periodic nx x ny grid, x fastest."""
    def nb(e, d, s):
        i, j = e % nx, e // nx
        if d == 0:
            i = (i + (1 if s else -1)) % nx
        else:
            j = (j + (1 if s else -1)) % ny
        return j * nx + i
    return nb


@pytest.mark.parametrize("system", ["euler", "navier-stokes"])
def test_p0_is_first_order_finite_volume(system):
    nx, ny, Lx, Ly = 4, 3, 2.0, 3.0
    hx, hy = Lx / nx, Ly / ny
    mesh = W.box_mesh((nx, ny), (Lx, Ly))
    prm = dict(p=0, system=system, gamma=G, mu=0.05, Pr=0.71, beta=0.5, tau=0.1)
    o = FROracle(mesh, prm)
    rng = np.random.default_rng(3)
    prim = np.stack([1 + rng.uniform(size=nx * ny), rng.uniform(-1, 1, nx * ny), rng.uniform(-1, 1, nx * ny), 1 + rng.uniform(size=nx * ny)])
    U = np.stack([prim[0], prim[0] * prim[1], prim[0] * prim[2], prim[3] / (G - 1) + 0.5 * prim[0] * (prim[1] ** 2 + prim[2] ** 2)])  # [4, Nel]
    R = o.rhs(U[None])[0]  # [NV, Nel]
    nb = _fv_neighbours(nx, ny)
    area = {0: hy, 1: hx}
    vol = hx * hy
    normal = {(0, 0): (-1.0, 0.0), (0, 1): (1.0, 0.0), (1, 0): (0.0, -1.0), (1, 1): (0.0, 1.0)}
    # hand-written cell-centred scheme.  Interface convention (A12): the low-side cell is L.
    q = np.zeros((nx * ny, 2, 4))
    if system == "navier-stokes":
        for e in range(nx * ny):
            for d in range(2):
                for s in range(2):
                    n = normal[(d, s)]
                    # beta = 1/2: common solution = u_R of the interface; at my high face (s=1) I am L
                    C = U[:, nb(e, d, 1)] if s == 1 else U[:, e]
                    for k in range(2):
                        q[e, k] += (C - U[:, e]) * n[k] * area[d] / vol
    expect = np.zeros_like(R)
    for e in range(nx * ny):
        for d in range(2):
            for s in range(2):
                o_ = nb(e, d, s)
                L, Rr = (e, o_) if s == 1 else (o_, e)
                nL = np.array(normal[(d, 1)])
                F = common_flux(U[:, L], U[:, Rr], q[L], q[Rr], nL, prm)
                sign = 1.0 if s == 1 else -1.0  # outward flux for cell e
                expect[:, e] -= sign * F * area[d] / vol
    assert np.allclose(R, expect, atol=1e-13, rtol=1e-13)


# ------------------------------------------------------------------------------------------
# the scheme converges spectrally to the analytic -div f (pins every term of Eq 20-24, the
# lifting scale factors, metric transforms and interface treatment at once)
# ------------------------------------------------------------------------------------------
def _analytic_ns_rhs(nd, mu, Pr):
    """-div(f_inv - f_vis) of Eq 20-24 by symbolic differentiation, with T = p/(rho R), R_gas = 1,
    C_p = g/(g-1) written explicitly (independent of the oracle's reduction A8)."""
    import sympy as sp

    xs = sp.symbols("x y z")[:nd]
    g = sp.Rational(7, 5)
    rho = 1 + sp.Rational(1, 5) * sp.sin(xs[0]) * sp.cos(xs[1]) * (sp.cos(xs[2]) if nd == 3 else 1)
    v = [sp.Rational(1, 2) + sp.Rational(3, 10) * sp.cos(xs[0]) * sp.sin(xs[1]), sp.Rational(-1, 4) + sp.Rational(1, 5) * sp.sin(xs[0] + xs[1])]
    if nd == 3:
        v.append(sp.Rational(1, 3) + sp.Rational(1, 4) * sp.sin(xs[2]) * sp.cos(xs[0]))
    p = 2 + sp.Rational(3, 10) * sp.cos(xs[0]) * sp.cos(xs[1]) * (sp.sin(xs[2]) if nd == 3 else 1)
    E = p / (g - 1) + rho * sum(c * c for c in v) / 2
    T = p / rho
    Cp = g / (g - 1)
    divv = sum(sp.diff(v[i], xs[i]) for i in range(nd))
    Tij = [[mu * (sp.diff(v[j], xs[i]) + sp.diff(v[i], xs[j])) - (sp.Rational(2, 3) * mu * divv if i == j else 0) for j in range(nd)] for i in range(nd)]
    U = [rho] + [rho * c for c in v] + [E]
    rhs = []
    for a in range(nd + 2):
        div = 0
        for n in range(nd):
            if a == 0:
                f = rho * v[n]
            elif a <= nd:
                j = a - 1
                f = rho * v[n] * v[j] + (p if j == n else 0) - Tij[n][j]
            else:
                f = v[n] * (E + p) - (sum(v[i] * Tij[i][n] for i in range(nd)) + mu * Cp / Pr * sp.diff(T, xs[n]))
            div += sp.diff(f, xs[n])
        rhs.append(-div)
    return sp.lambdify(xs, U, "numpy"), sp.lambdify(xs, rhs, "numpy")


@pytest.mark.parametrize("kind", ["hex", "quad-curved", "tri"])
def test_rhs_converges_to_analytic_navier_stokes(kind):
    mu, Pr = 0.05, 0.71
    nd = 3 if kind == "hex" else 2
    fU, fR = _analytic_ns_rhs(nd, mu, Pr)
    errs = []
    orders = (3, 6, 9) if kind != "hex" else (3, 5, 7)
    for p in orders:
        if kind == "hex":
            mesh = W.box_mesh((3, 3, 3), (2 * np.pi,) * 3)
        elif kind == "quad-curved":
            mesh = W.box_mesh((4, 4), (2 * np.pi,) * 2, p_g=2, warp=lambda X: 0.1 * np.stack([np.sin(X[..., 0]) * np.sin(X[..., 1]), -np.sin(X[..., 0]) * np.sin(X[..., 1])], -1))
        else:
            mesh = W.tri_mesh(8, 2 * np.pi, 0.1, 7)
        o = FROracle(mesh, dict(p=p, system="navier-stokes", gamma=G, mu=mu, Pr=Pr, beta=0.5, tau=0.1))
        X = _coords(o)
        args = [X[..., d] for d in range(nd)]
        U = np.stack([np.broadcast_to(a, X.shape[:-1]) for a in fU(*args)], 1)
        exact = np.stack([np.broadcast_to(a, X.shape[:-1]) for a in fR(*args)], 1)
        R = o.rhs(U)
        errs.append(np.max(np.abs(R - exact) / np.max(np.abs(exact), axis=(0, 2))[None, :, None]))
    assert errs[0] > errs[1] > errs[2]
    assert errs[-1] < (2e-3 if kind == "hex" else 2e-4), errs
    assert errs[0] / errs[-1] > 50, errs


# ------------------------------------------------------------------------------------------
# freestream preservation and discrete conservation (north_star pins 3, 4)
# ------------------------------------------------------------------------------------------
MESHES = {
    "quad-affine": lambda p: W.box_mesh((5, 4), (10.0, 7.0)),
    "quad-curved": lambda p: W.box_mesh((4, 4), (2 * np.pi,) * 2, p_g=min(p, 3), warp=lambda X: 0.08 * np.stack([np.sin(X[..., 0]) * np.sin(X[..., 1]), np.sin(2 * X[..., 0]) * np.sin(X[..., 1])], -1)),
    "hex-affine": lambda p: W.box_mesh((3, 3, 3), (2 * np.pi,) * 3),
    "hex-curved": lambda p: W.box_mesh((3, 3, 3), (2 * np.pi,) * 3, p_g=p, warp=W.sine_warp(0.05)),
    "tri-jitter": lambda p: W.tri_mesh(6, 1.0, 0.1, 4321),
}


@pytest.mark.parametrize("name,p", [("quad-affine", 2), ("quad-curved", 3), ("hex-affine", 2), ("hex-curved", 3), ("tri-jitter", 3)])
@pytest.mark.parametrize("system", ["euler", "navier-stokes"])
def test_freestream_and_conservation(name, p, system):
    mesh = MESHES[name](p)
    o = FROracle(mesh, dict(p=p, system=system, gamma=G, mu=0.02, Pr=0.71, beta=0.5, tau=0.1))
    nd = o.nd
    h = min(mesh["lengths"]) / max(mesh["shape"])
    U0 = _state_on(o, W.uniform_state, rho=1.0, vel=(1.0, 0.5, 0.25)[:nd], p=1.0)
    fmax = np.max(np.abs(flux_inviscid(np.moveaxis(U0, 1, 0), G)))
    assert np.max(np.abs(o.rhs(U0))) <= 1e-12 * fmax * 2 / h
    # noisy smooth state: quadrature- and |J|-weighted sum of the RHS vanishes
    X = _coords(o)
    fn = W.taylor_green if nd == 3 else (lambda X: W.sinusoidal_2d(X / max(mesh["lengths"])))
    U = np.moveaxis(W.add_relative_noise(fn(X), 1e-2, 11), -1, 1)
    R = o.rhs(U)
    assert np.all(np.abs(o.integrate(R)) <= 1e-12 * o.integrate(np.abs(R)))
    assert np.all(o.integrate(np.abs(R)) > 1e-3)


# ------------------------------------------------------------------------------------------
# order of accuracy p+1 for the isentropic vortex (north_star pin 5)
# ------------------------------------------------------------------------------------------
@pytest.mark.parametrize("p", [1, 2, 3])
def test_vortex_order_of_accuracy(p):
    errs, hs = [], []
    t_end = 0.2
    for n in (8, 16, 32):
        mesh = W.box_mesh((n, n), (10.0, 10.0))
        o = FROracle(mesh, dict(p=p, system="euler", gamma=G, mu=0.0, Pr=0.71, beta=0.5, tau=0.0))
        U = _state_on(o, W.isentropic_vortex)
        steps = int(np.ceil(t_end / (0.1 * (10.0 / n) / (2 * p + 1) / 3.0)))
        dt = t_end / steps
        for _ in range(steps):
            U = o.rk4_step(U, dt)
        exact = _state_on(o, W.isentropic_vortex, t=t_end, period=10.0)
        errs.append(o.l2_error(U, exact)[0])
        hs.append(10.0 / n)
    slope = np.polyfit(np.log(hs), np.log(errs), 1)[0]
    assert p + 0.6 < slope < p + 2.2, (slope, errs)


def test_rk4_stability_polynomial():
    """Classical RK4 on u' = lambda u multiplies by 1 + z + z^2/2 + z^3/6 + z^4/24 exactly (:247)."""
    mesh = W.box_mesh((2, 2), (1.0, 1.0))
    o = FROracle(mesh, dict(p=1, system="euler", gamma=G, mu=0.0, Pr=0.71, beta=0.5, tau=0.0))
    lam, dt = -1.3, 0.37
    o.rhs = lambda u: lam * u
    u0 = np.random.default_rng(0).standard_normal((4, 4, 4))
    z = lam * dt
    assert np.allclose(o.rk4_step(u0, dt), u0 * (1 + z + z * z / 2 + z ** 3 / 6 + z ** 4 / 24), rtol=1e-14)
    # order: error of one step on u' = u vs exp(dt) is ~dt^5/120
    o.rhs = lambda u: u
    e1 = abs(o.rk4_step(np.ones(1), 0.1)[0] - np.exp(0.1))
    e2 = abs(o.rk4_step(np.ones(1), 0.05)[0] - np.exp(0.05))
    assert 28 < e1 / e2 < 36


# ------------------------------------------------------------------------------------------
# boundary conditions (Appendix C) and the paper's Couette case (Eq 34-36, constants at :589)
# ------------------------------------------------------------------------------------------
def test_characteristic_boundaries_preserve_matching_freestream():
    mesh = W.box_mesh((3, 3), (1.0, 1.0), periodic=False)
    free = dict(rho=1.2, v=(2.5, 0.4), p=1.0)  # supersonic in x
    bcs = {0: ("sup-inflow", free), 1: ("sub-outflow", dict(p=1.0)), 2: ("sup-inflow", free), 3: ("sub-outflow", dict(p=1.0))}
    for system in ("euler", "navier-stokes"):
        o = FROracle(mesh, dict(p=2, system=system, gamma=G, mu=0.01, Pr=0.71, beta=0.5, tau=0.1), bcs)
        U = _state_on(o, W.uniform_state, rho=1.2, vel=(2.5, 0.4), p=1.0)
        assert np.max(np.abs(o.rhs(U))) < 1e-11


def couette_state(X, gamma=1.4, Pr=0.72, cp=1005.0, Tw=300.0, pc=1e5, vw=69.445, H=1.0):
    """PAPER.md:580-589 Eq 34-36 with the constants printed at :589."""
    phi = X[..., 1] / H
    rho = gamma / (gamma - 1) * 2 * pc / (2 * cp * Tw + Pr * vw * vw * phi * (1 - phi))
    u = vw * phi
    return np.stack([rho, rho * u, 0 * rho, pc / (gamma - 1) + 0.5 * rho * u * u], -1)


def test_couette_is_a_steady_state_with_wall_bcs():
    """The paper's analytic Couette solution is steady: RHS -> 0 spectrally in p with the no-slip
    isothermal wall BCs of App C.4 (bottom wall at rest, top wall moving at v_w)."""
    cp, Tw, vw, Pr, mu = 1005.0, 300.0, 69.445, 0.72, 0.417
    mesh = W.box_mesh((2, 2), (1.0, 1.0), periodic=(True, False))
    bcs = {2: ("noslip-wall", dict(cpTw=cp * Tw, v=(0.0, 0.0))), 3: ("noslip-wall", dict(cpTw=cp * Tw, v=(vw, 0.0)))}
    res = []
    for p in (1, 2, 4):
        o = FROracle(mesh, dict(p=p, system="navier-stokes", gamma=G, mu=mu, Pr=Pr, beta=0.5, tau=0.1), bcs)
        U = _state_on(o, couette_state)
        R = o.rhs(U)
        # scale: momentum-flux magnitude p_c times 2/h
        res.append(np.max(np.abs(R[:, 1:3])) / (1e5 * 2 / 0.5))
    assert res[0] > 10 * res[1] > 100 * res[2] and res[2] < 1e-7, res
