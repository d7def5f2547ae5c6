"""Pins for the oracle's point-wise physics (O8, O9, Appendix B/C): hand-worked numbers,
closed forms and the invariants the paper states."""
import numpy as np
import pytest

from oracle.fr_oracle import common_flux, flux_inviscid, flux_viscous, ghost_states, ldg_viscous, rusanov

G = 1.4


def _state(rho, v, p):
    v = list(v)
    return np.array([rho] + [rho * x for x in v] + [p / (G - 1) + 0.5 * rho * sum(x * x for x in v)], dtype=float)


def test_euler_flux_hand_values_3d():
    """Eq 20-21 (:474-481) evaluated by hand for rho=2, v=(3,4,5), p=7:
    E = 7/0.4 + 0.5*2*50 = 67.5; E+p = 74.5."""
    u = _state(2.0, (3.0, 4.0, 5.0), 7.0)
    assert u[4] == pytest.approx(67.5, abs=1e-13)
    f = flux_inviscid(u, G)
    expect = np.array(
        [
            [6.0, 18.0 + 7.0, 24.0, 30.0, 3 * 74.5],
            [8.0, 24.0, 32.0 + 7.0, 40.0, 4 * 74.5],
            [10.0, 30.0, 40.0, 50.0 + 7.0, 5 * 74.5],
        ]
    )
    assert np.allclose(f, expect, atol=1e-12)


def test_euler_flux_2d_reduction():
    """:520 — delete the 4th row and 3rd column."""
    u3 = _state(2.0, (3.0, 4.0, 0.0), 7.0)
    u2 = _state(2.0, (3.0, 4.0), 7.0)
    f3, f2 = flux_inviscid(u3, G), flux_inviscid(u2, G)
    assert np.allclose(f2, f3[:2][:, [0, 1, 2, 4]], atol=1e-13)


def _grad_from_primitive(rho, v, p, drho, dv, dp):
    """gradient of the conserved variables from primitive gradients (product rule), dv[i][j] = d_i v_j."""
    nd = len(v)
    q = np.zeros((nd, nd + 2))
    for i in range(nd):
        q[i, 0] = drho[i]
        for j in range(nd):
            q[i, 1 + j] = drho[i] * v[j] + rho * dv[i][j]
        q[i, nd + 1] = dp[i] / (G - 1) + 0.5 * drho[i] * sum(x * x for x in v) + rho * sum(v[j] * dv[i][j] for j in range(nd))
    return q


def test_viscous_pure_shear():
    """Eq 23 (:494): v = (a*y, 0, 0) at uniform rho, p  =>  only T_xy = T_yx = mu*a."""
    mu, a = 0.3, 1.7
    rho, v, p = 1.3, (0.4, 0.0, 0.0), 2.0
    dv = [[0.0] * 3 for _ in range(3)]
    dv[1][0] = a  # d_y v_x
    q = _grad_from_primitive(rho, v, p, [0] * 3, dv, [0] * 3)
    f = flux_viscous(_state(rho, v, p), q, G, mu, 0.71)
    expect = np.zeros((3, 5))
    expect[1, 1] = mu * a  # direction y, x-momentum: T_yx
    expect[0, 2] = mu * a  # direction x, y-momentum: T_xy
    expect[1, 4] = v[0] * mu * a  # v_i T_iy = v_x T_xy
    assert np.allclose(f, expect, atol=1e-14)


def test_viscous_uniform_dilatation_3d_and_2d():
    """3-D: trace-free => T == 0.  2-D keeps the 2/3 (reading A22): T_ii = 2 mu a - (2/3) mu 2a = (2/3) mu a."""
    mu, a = 0.3, 1.7
    for nd in (3, 2):
        v = (0.0,) * nd
        dv = [[a if i == j else 0.0 for j in range(nd)] for i in range(nd)]
        q = _grad_from_primitive(1.3, v, 2.0, [0] * nd, dv, [0] * nd)
        f = flux_viscous(_state(1.3, v, 2.0), q, G, mu, 0.71)
        expect = np.zeros((nd, nd + 2))
        if nd == 2:
            expect[0, 1] = expect[1, 2] = 2.0 / 3.0 * mu * a
        assert np.allclose(f, expect, atol=1e-14)


def test_viscous_heat_flux():
    """Eq 22, 24 (:489-500) with explicit C_p, C_v (R_gas = 1 => C_v = 1/(g-1), C_p = g/(g-1)):
    fluid at rest, uniform rho, dp/dx = b  =>  T = p/(rho R), energy flux_x = (mu C_p/Pr) dT/dx."""
    mu, Pr, b, rho, p = 0.3, 0.71, 0.9, 1.3, 2.0
    q = _grad_from_primitive(rho, (0, 0, 0), p, [0] * 3, [[0] * 3] * 3, [b, 0, 0])
    f = flux_viscous(_state(rho, (0, 0, 0), p), q, G, mu, Pr)
    Cp = G / (G - 1)
    expect = np.zeros((3, 5))
    expect[0, 4] = mu * Cp / Pr * (b / rho)
    assert np.allclose(f, expect, atol=1e-14)
    # density gradient at constant p: dT/dx = -p/(rho^2) drho/dx
    q = _grad_from_primitive(rho, (0, 0, 0), p, [b, 0, 0], [[0] * 3] * 3, [0, 0, 0])
    f = flux_viscous(_state(rho, (0, 0, 0), p), q, G, mu, Pr)
    assert f[0, 4] == pytest.approx(mu * Cp / Pr * (-p / rho ** 2 * b), abs=1e-14)


def test_rusanov_hand_values():
    """Eq 45-46 (:785-789), fluid at rest on both sides, n = x:
    s = sqrt(g (pL+pR)/(rL+rR)); F = (s/2 (rL-rR), (pL+pR)/2, 0, 0, s/2 (EL-ER))."""
    uL, uR = _state(1.0, (0, 0, 0), 1.0), _state(0.5, (0, 0, 0), 0.25)
    n = np.array([1.0, 0.0, 0.0])
    s = np.sqrt(G * 1.25 / 1.5)
    F = rusanov(uL, uR, n, G)
    assert np.allclose(F, [s / 2 * 0.5, 0.625, 0, 0, s / 2 * (1.0 - 0.25) / (G - 1)], atol=1e-14)
    # moving: the |n.(vL+vR)|/2 term of the printed Eq 46 (reading A14)
    uL, uR = _state(1.0, (0.3, 0, 0), 1.0), _state(1.0, (0.5, 0, 0), 1.0)
    F = rusanov(uL, uR, n, G)
    s = np.sqrt(G * 2 / 2) + 0.5 * 0.8
    central_rho = 0.5 * (0.3 + 0.5)
    assert F[0] == pytest.approx(central_rho + s / 2 * 0.0, abs=1e-14)
    assert F[1] == pytest.approx(0.5 * (0.09 + 1 + 0.25 + 1) + s / 2 * (0.3 - 0.5), abs=1e-14)


def _rand_states(nd, seed):
    rng = np.random.default_rng(seed)
    mk = lambda: _state(1 + rng.uniform(), rng.uniform(-1, 1, nd), 1 + rng.uniform())
    n = rng.standard_normal(nd)
    return mk(), mk(), rng.standard_normal((nd, nd + 2)), rng.standard_normal((nd, nd + 2)), n / np.linalg.norm(n)


@pytest.mark.parametrize("nd", [2, 3])
@pytest.mark.parametrize("system", ["euler", "navier-stokes"])
def test_common_flux_consistency_and_antisymmetry(nd, system):
    """F(u,u,q,q,n) = n.f(u,q); F(L,R,n) = -F(R,L,-n) with beta -> -beta (:229); C(u,u) = u."""
    uL, uR, qL, qR, n = _rand_states(nd, 5)
    prm = dict(system=system, gamma=G, mu=0.2, Pr=0.71, beta=0.5, tau=0.1)
    f = flux_inviscid(uL, G) - (flux_viscous(uL, qL, G, 0.2, 0.71) if system != "euler" else 0)
    assert np.allclose(common_flux(uL, uL, qL, qL, n, prm), np.einsum("d,dv->v", n, f), atol=1e-13)
    for beta in (0.5, 0.0, -0.3):
        a = common_flux(uL, uR, qL, qR, n, dict(prm, beta=beta))
        b = common_flux(uR, uL, qR, qL, -n, dict(prm, beta=-beta))
        assert np.allclose(a, -b, atol=1e-13)


def test_ldg_upwinding_direction():
    """Eq 25/27 (:506-514): beta=+1/2 takes the common SOLUTION from R and the viscous FLUX from L."""
    uL, uR, qL, qR, n = _rand_states(3, 7)
    Fv = ldg_viscous(uL, uR, qL, qR, n, G, 0.2, 0.71, 0.5, 0.0)
    assert np.allclose(Fv, np.einsum("d,dv->v", n, flux_viscous(uL, qL, G, 0.2, 0.71)), atol=1e-14)
    Fv = ldg_viscous(uL, uR, qL, qR, n, G, 0.2, 0.71, -0.5, 0.0)
    assert np.allclose(Fv, np.einsum("d,dv->v", n, flux_viscous(uR, qR, G, 0.2, 0.71)), atol=1e-14)


def test_penalty_is_dissipative():
    """Reading A7: the tau jump term has the sign of Rusanov's s/2 (u_L - u_R) term."""
    uL, uR, qL, qR, n = _rand_states(3, 9)
    prm = dict(system="navier-stokes", gamma=G, mu=0.2, Pr=0.71, beta=0.5, tau=0.0)
    d = common_flux(uL, uR, qL, qR, n, dict(prm, tau=0.25)) - common_flux(uL, uR, qL, qR, n, prm)
    assert np.allclose(d, 0.25 * (uL - uR), atol=1e-13)


def test_ghost_states_hand_values():
    """Appendix C Eq 47-53 (:801-825) for rho_L=2, v_L=(3,4), p_L=7."""
    uL = _state(2.0, (3.0, 4.0), 7.0)[:, None]
    gi, gl, keep = ghost_states("sup-inflow", dict(rho=1.5, v=(2.0, 0.5), p=3.0), uL, G)
    e = 3.0 / 0.4 + 0.75 * (4 + 0.25)
    assert np.allclose(gi[:, 0], [1.5, 3.0, 0.75, e]) and np.allclose(gl, gi) and keep == 0.0
    gi, gl, keep = ghost_states("sub-outflow", dict(p=3.0), uL, G)
    assert np.allclose(gi[:, 0], [2.0, 6.0, 8.0, 3.0 / 0.4 + 25.0]) and np.allclose(gl, gi) and keep == 0.0
    gi, gl, keep = ghost_states("noslip-wall", dict(cpTw=10.0, v=(1.0, 0.0)), uL, G)
    # B_inv: velocity 2 v_w - v_L = (-1, -4); B_ldg: velocity v_w
    assert np.allclose(gi[:, 0], [2.0, -2.0, -8.0, 2.0 * (10.0 / 1.4 + 0.5 * 17.0)])
    assert np.allclose(gl[:, 0], [2.0, 2.0, 0.0, 2.0 * (10.0 / 1.4 + 0.5)])
    assert keep == 1.0
