"""Pins for the oracle's other FR schemes (SD / HU correction functions) and time steppers (Euler, DOPRI5,
Table 1 :263).  The expected values are closed-form properties from the literature the paper cites, order conditions of
Runge-Kutta theory and stability polynomials -- none re-uses the oracle's formulas."""
import math

import numpy as np
import pytest
from numpy.polynomial import legendre as npleg

import workloads as W
from oracle.fr_oracle import (DOPRI5_A, DOPRI5_B4, DOPRI5_B5, LD, FROracle, Operators, RefElement, correction_derivative_1d,
                              gauss_legendre)


def _g_at(scheme, p, x):
    """g_R(x) = integral of the oracle's g_R' from -1 to x (Gauss quadrature, exact for the degree-p integrand)."""
    t, w = gauss_legendre(p + 2)
    x = LD(x)
    s = (x + 1) / 2 * (t + 1) - 1  # [-1, x]
    return float(np.sum(w * correction_derivative_1d(scheme, p, s)) * (x + 1) / 2)


@pytest.mark.parametrize("p", [1, 2, 3, 4, 5])
def test_correction_functions_closed_form_properties(p):
    unit = np.zeros(p + 1)
    unit[p] = 1
    gauss_p = npleg.legroots(unit)                    # roots of P_p
    lobatto_int = npleg.legroots(npleg.legder(unit))  # roots of P_p': interior points of the (p+1)-point Gauss-Lobatto rule
    radau = npleg.legroots(np.r_[np.zeros(p), 1.0, 1.0])  # roots of P_p + P_{p+1} (right Radau polynomial of degree p+1)
    for scheme in ("dg", "sd", "hu"):
        assert abs(_g_at(scheme, p, 1.0) - 1.0) < 1e-14, scheme  # g_R(1) - g_R(-1) = 1
    # DG: g_R is the right Radau polynomial: zero at all its p+1 roots (-1 among them)
    assert max(abs(_g_at("dg", p, r)) for r in radau) < 1e-13
    # SD: g_R vanishes at the p Gauss points (the flux points of the spectral difference scheme it recovers)
    assert max(abs(_g_at("sd", p, r)) for r in gauss_p) < 1e-13
    assert max(abs(_g_at("dg", p, r)) for r in gauss_p) > 1e-3  # and that distinguishes it from DG
    # HU (Huynh's g_2): g_R' vanishes at the interior Gauss-Lobatto points and at -1
    d = np.asarray(correction_derivative_1d("hu", p, np.r_[lobatto_int, -1.0]), float)
    assert np.max(np.abs(d)) < 1e-12
    assert abs(float(correction_derivative_1d("sd", p, np.array([-1.0]))[0])) > 1e-3
    # stiffness ordering c_DG < c_SD < c_HU: the end slope g_R'(1) decreases along the family; DG's is (p+1)^2 / 2
    s = [float(correction_derivative_1d(k, p, np.array([1.0]))[0]) for k in ("dg", "sd", "hu")]
    assert s[0] > s[1] > s[2] > 0
    assert abs(s[0] - (p + 1) ** 2 / 2) < 1e-12


@pytest.mark.parametrize("etype,p,scheme", [("quad", 2, "sd"), ("quad", 3, "hu"), ("hex", 2, "hu"), ("hex", 1, "sd")])
def test_sd_hu_operators_keep_the_conservation_identities(etype, p, scheme):
    """w^T M3 = w^f and w^T (M1 - M3 M2) = 0 (discrete divergence theorem) hold for every member of the family, because
    int g_R' = 1 and the quadrature is exact for degree p; M3 differs from DG's."""
    ref = RefElement(etype, p)
    o, dg = Operators(ref, scheme), Operators(ref)
    w = ref.wu
    assert np.max(np.abs(w @ o.M3 - ref.wf)) < 1e-15
    assert np.max(np.abs(w @ (o.M1 - o.M3 @ o.M2))) < 1e-14
    assert np.max(np.abs(o.M3 - dg.M3)) > 1e-2
    assert np.allclose(np.asarray(o.M0, float), np.asarray(dg.M0, float))


def test_sd_hu_are_rejected_on_triangles():
    with pytest.raises(ValueError):
        Operators(RefElement("tri", 2), "sd")


@pytest.mark.parametrize("scheme", ["sd", "hu"])
def test_sd_hu_freestream_conservation_and_vortex_order(scheme):
    mesh, disc = W.config("C3", n=2, p=2)
    disc = dict(disc, correction=scheme)
    o = FROracle(mesh, disc)
    X = np.asarray(o.xu_phys, float)
    U0 = np.moveaxis(W.uniform_state(X, rho=1.0, vel=(1.0, 1.0, 1.0), p=1.0), -1, 1)
    assert np.max(np.abs(o.rhs(U0))) < 1e-11
    U = W.config_state("C3", X, n=2, p=2)
    R = o.rhs(U)
    assert np.all(np.abs(o.integrate(R)) <= 1e-12 * o.integrate(np.abs(R)))
    assert np.max(np.abs(R - FROracle(mesh, dict(disc, correction="dg")).rhs(U))) > 1e-6 * np.max(np.abs(R))
    # isentropic vortex, p = 2: L2 density error of the semi-discrete RHS against the exact time derivative ~ h^p at least
    errs = []
    for n in (8, 16):
        m = W.box_mesh((n, n), (10.0, 10.0))
        d = dict(p=2, system="euler", gamma=1.4, mu=0.0, Pr=0.71, beta=0.5, tau=0.0, correction=scheme)
        ov = FROracle(m, d)
        Xv = np.asarray(ov.xu_phys, float)
        dt = 1e-4
        exact = (W.isentropic_vortex(Xv, dt, period=10.0) - W.isentropic_vortex(Xv, -dt, period=10.0)) / (2 * dt)
        Rv = ov.rhs(np.ascontiguousarray(np.moveaxis(W.isentropic_vortex(Xv), -1, 1)))
        errs.append(float(ov.l2_error(Rv, np.moveaxis(exact, -1, 1))[0]))
    assert np.log2(errs[0] / errs[1]) > 1.7, errs


# ----------------------------------------------------------------------------------------------
# time steppers
# ----------------------------------------------------------------------------------------------
def test_dopri5_tableau_order_conditions():
    """Row sums give the nodes c = (0, 1/5, 3/10, 4/5, 8/9, 1, 1); the weights b5 satisfy all 17 rooted-tree order conditions
    to order 5, b4 those to order 4 and not order 5; the 7th row of A equals b5 (first-same-as-last)."""
    A = np.zeros((7, 7))
    for i, row in enumerate(DOPRI5_A):
        A[i, : len(row)] = row
    c = A.sum(1)
    assert np.allclose(c, [0, 1 / 5, 3 / 10, 4 / 5, 8 / 9, 1, 1], atol=1e-15)
    assert np.allclose(A[6, :6], DOPRI5_B5[:6], atol=0) and DOPRI5_B5[6] == 0
    Ac, Ac2, Ac3, AAc = A @ c, A @ c ** 2, A @ c ** 3, A @ (A @ c)
    conds = [  # (elementary weight vector, 1/gamma(tree))
        (np.ones(7), 1), (c, 1 / 2), (c ** 2, 1 / 3), (Ac, 1 / 6),
        (c ** 3, 1 / 4), (c * Ac, 1 / 8), (Ac2, 1 / 12), (AAc, 1 / 24),
        (c ** 4, 1 / 5), (c ** 2 * Ac, 1 / 10), (c * Ac2, 1 / 15), (c * AAc, 1 / 30), (Ac ** 2, 1 / 20), (Ac3, 1 / 20),
        (A @ (c * Ac), 1 / 40), (A @ Ac2, 1 / 60), (A @ AAc, 1 / 120),
    ]
    b5, b4 = np.array(DOPRI5_B5), np.array(DOPRI5_B4)
    r5 = [abs(b5 @ phi - g) for phi, g in conds]
    r4 = [abs(b4 @ phi - g) for phi, g in conds]
    assert max(r5) < 1e-15, r5
    assert max(r4[:8]) < 1e-15 and max(r4[8:]) > 1e-4, r4


class _Linear(FROracle):
    """u' = lam u through the oracle's stepper code (rhs replaced, steppers untouched)."""

    def __init__(self, lam):
        self.lam = lam

    def rhs(self, u, return_parts=False):
        return self.lam * u


def test_stepper_stability_polynomials():
    """One step of u' = lam u multiplies u by the scheme's stability polynomial: Euler 1 + z; DOPRI5
    sum_{k<=5} z^k / k! + z^6 / 600; its embedded error estimate is O(z^5)."""
    u = np.array([[[1.0]]])
    for z in (0.1, -0.7, 0.3 + 0.4j):
        o = _Linear(z)
        assert abs(o.euler_step(u.astype(complex), 1.0)[0, 0, 0] - (1 + z)) < 1e-15
        new, err = o.dopri5_step(u.astype(complex), 1.0)
        want = sum(z ** k / math.factorial(k) for k in range(6)) + z ** 6 / 600
        assert abs(new[0, 0, 0] - want) < 1e-15
    e1 = abs(_Linear(0.1).dopri5_step(u, 1.0)[1][0, 0, 0])
    e2 = abs(_Linear(0.05).dopri5_step(u, 1.0)[1][0, 0, 0])
    assert 4.7 < np.log2(e1 / e2) < 5.3  # leading error term z^5


def test_dopri5_converges_at_fifth_order_on_the_vortex():
    mesh, disc = W.config("C1")
    o = FROracle(mesh, disc)
    U = W.config_state("C1", np.asarray(o.xu_phys, float))
    T = 0.08
    ref = U
    for _ in range(16):
        ref, _ = o.dopri5_step(ref, T / 16)
    errs = []
    for n in (1, 2):
        u = U
        for _ in range(n):
            u, _ = o.dopri5_step(u, T / n)
        errs.append(np.max(np.abs(u - ref)))
    assert np.log2(errs[0] / errs[1]) > 4.3, errs
