"""Pins for the oracle's O1-O3 (quadrature, nodal bases, operator matrices M0..M6).
Each test cites what fixes the expected value; none re-uses the oracle's own formula."""
import itertools

import numpy as np
import pytest

from oracle.fr_oracle import LD, Operators, RefElement, gauss_legendre, lagrange_1d

ETYPES = [("quad", 1), ("quad", 2), ("quad", 4), ("hex", 1), ("hex", 3), ("tri", 1), ("tri", 2), ("tri", 3), ("tri", 4)]


def _load_golden():
    import os

    out = {}
    with open(os.path.join(os.path.dirname(__file__), "golden", "gauss_legendre_closed_forms.txt")) as f:
        for line in f:
            if line.startswith("#") or not line.strip():
                continue
            n, kind, vals = line.split(";")
            out[(int(n), kind.strip())] = [float(eval(v, {"sqrt": np.sqrt})) for v in vals.split(",")]
    return out


def test_gauss_legendre_closed_forms():
    """Textbook closed forms n=1,2,3 (tests/golden/gauss_legendre_closed_forms.txt)."""
    gold = _load_golden()
    for n in (1, 2, 3):
        x, w = gauss_legendre(n)
        assert np.allclose(np.asarray(x, float), gold[(n, "x")], atol=2.3e-16, rtol=0)
        assert np.allclose(np.asarray(w, float), gold[(n, "w")], atol=2.3e-16, rtol=0)


@pytest.mark.parametrize("n", range(1, 9))
def test_gauss_legendre_exactness(n):
    """n-point GL integrates x^k exactly for k <= 2n-1: integral = 2/(k+1) (k even), 0 (odd)."""
    x, w = gauss_legendre(n)
    assert abs(float(w.sum()) - 2.0) < 1e-17
    for k in range(2 * n):
        exact = 2.0 / (k + 1) if k % 2 == 0 else 0.0
        assert abs(float(np.sum(w * x ** k)) - exact) < 1e-17
    # and is NOT exact for degree 2n (guards against an off-by-one node count)
    assert abs(float(np.sum(w * x ** (2 * n))) - 2.0 / (2 * n + 1)) > 1e-8


def test_lagrange_cardinal_and_derivative():
    """l_j(x_i) = delta_ij; derivative of the interpolant of x^k is k x^(k-1)."""
    nodes, _ = gauss_legendre(5)
    L, dL = lagrange_1d(nodes, nodes)
    assert np.allclose(np.asarray(L, float), np.eye(5), atol=1e-17)
    x = np.linspace(-1, 1, 7)
    L, dL = lagrange_1d(nodes, x)
    for k in range(5):
        assert np.allclose(np.asarray(L @ nodes ** k, float), x ** k, atol=1e-16)
        assert np.allclose(np.asarray(dL @ nodes ** k, float), k * x ** max(k - 1, 0) if k else 0 * x, atol=1e-15)


def _monomials(nd, p, etype):
    if etype == "tri":
        return [e for e in itertools.product(range(p + 1), repeat=2) if sum(e) <= p]
    return list(itertools.product(range(p + 1), repeat=nd))


def _mono(X, e):
    return np.prod([X[:, d] ** e[d] for d in range(len(e))], axis=0)


def _dmono(X, e, dd):
    if e[dd] == 0:
        return np.zeros(X.shape[0], dtype=X.dtype)
    f = [X[:, d] ** (e[d] - 1 if d == dd else e[d]) for d in range(len(e))]
    return e[dd] * np.prod(f, axis=0)


@pytest.mark.parametrize("etype,p", ETYPES)
def test_point_counts_and_cardinality(etype, p):
    """Point counts (SURVEY notation) and l_rho(x_sigma) = delta."""
    ref = RefElement(etype, p)
    n = p + 1
    assert ref.Nu == {"quad": n * n, "hex": n ** 3, "tri": n * (n + 1) // 2}[etype]
    assert ref.Nf == {"quad": 4 * n, "hex": 6 * n * n, "tri": 3 * n}[etype]
    L, _ = ref.basis(ref.xu)
    assert np.allclose(np.asarray(L, float), np.eye(ref.Nu), atol=1e-15)
    # flux points lie on the boundary with unit outward normals
    assert np.allclose(np.asarray(np.sum(ref.nf ** 2, -1), float), 1.0, atol=1e-17)
    if etype == "tri":  # S3 symmetry of the solution point set (reading A6)
        lam = np.stack([(ref.xu[:, 0] + 1) / 2, (ref.xu[:, 1] + 1) / 2], -1)
        lam = np.concatenate([lam, 1 - lam.sum(-1, keepdims=True)], -1).astype(float)
        pts = {tuple(np.round(r, 12)) for r in lam}
        for perm in itertools.permutations(range(3)):
            assert {tuple(np.round(r[list(perm)], 12)) for r in lam} == pts


@pytest.mark.parametrize("etype,p", ETYPES)
def test_M0_M4_M1_polynomial_exactness(etype, p):
    """M0 reproduces, and M4 / M1 differentiate, every monomial of degree <= p exactly
    (north_star pin 1); M1 applied to a constant vector flux is zero (pin 2)."""
    ref = RefElement(etype, p)
    ops = Operators(ref)
    nd, Nu = ref.nd, ref.Nu
    for e in _monomials(nd, p, etype):
        uu = _mono(ref.xu, e)
        assert np.allclose(np.asarray(ops.M0 @ uu, float), np.asarray(_mono(ref.xf, e), float), atol=2e-15)
        g = (ops.M4 @ uu).reshape(nd, Nu)
        for d in range(nd):
            assert np.allclose(np.asarray(g[d], float), np.asarray(_dmono(ref.xu, e, d), float), atol=5e-14)
        # divergence of the vector field (x^e, 2 x^e, 3 x^e)
        F = np.concatenate([(d + 1) * uu for d in range(nd)])
        div = sum((d + 1) * _dmono(ref.xu, e, d) for d in range(nd))
        assert np.allclose(np.asarray(ops.M1 @ F, float), np.asarray(div, float), atol=1e-13)
    const = np.concatenate([np.full(Nu, LD(d + 2)) for d in range(nd)])
    assert np.max(np.abs(ops.M1 @ const)) < 1e-15
    assert np.allclose(np.asarray(ops.M0.sum(1), float), 1.0, atol=1e-15)  # partition of unity


@pytest.mark.parametrize("etype,p", ETYPES)
def test_M2_is_normal_trace(etype, p):
    """Eq 13 (:218): M2 F = n . (interpolated F) at the flux points, for polynomial F."""
    ref = RefElement(etype, p)
    ops = Operators(ref)
    nd = ref.nd
    e = _monomials(nd, p, etype)[-1]
    F = np.concatenate([(d + 1) * _mono(ref.xu, e) for d in range(nd)])
    expect = sum((d + 1) * _mono(ref.xf, e) * ref.nf[:, d] for d in range(nd))
    assert np.allclose(np.asarray(ops.M2 @ F, float), np.asarray(expect, float), atol=1e-14)


@pytest.mark.parametrize("etype,p", ETYPES)
def test_M3_divergence_theorem_and_conservation_identities(etype, p):
    """integral(div g_sigma) = boundary integral of n.g_sigma = w^f_sigma (Eq 8 :198 + GL face
    quadrature), i.e. w^T M3 = w^f; and w^T (M1 - M3 M2) = 0 (discrete conservation)."""
    ref = RefElement(etype, p)
    ops = Operators(ref)
    w = ref.wu
    vol = {"quad": 4.0, "hex": 8.0, "tri": 2.0}[etype]
    assert abs(float(w.sum()) - vol) < 1e-15
    assert np.allclose(np.asarray(w @ ops.M3, float), np.asarray(ref.wf, float), atol=1e-15)
    assert np.max(np.abs(np.asarray(w @ (ops.M1 - ops.M3 @ ops.M2), float))) < 1e-14


@pytest.mark.parametrize("etype,p", [("quad", 1), ("quad", 3), ("hex", 2), ("hex", 4)])
def test_M3_equals_radau_closed_form(etype, p):
    """DG correction on tensor elements = right Radau polynomial g_R = (-1)^p (P_p - P_{p+1})/2 ... in
    the form g_R(xi) = (P_p(xi) + P_{p+1}(xi))/2 for the +1 face, g_L(xi) = g_R(-xi) (Huynh's DG
    recovery, reading A5): div g_sigma is g' along the line through sigma, zero off the line."""
    from numpy.polynomial import legendre as NL

    ref = RefElement(etype, p)
    ops = Operators(ref)
    n, nd = p + 1, ref.nd
    g = np.asarray(ref.g1, float)
    cR = np.zeros(p + 2)
    cR[p], cR[p + 1] = 0.5, 0.5
    dgR = NL.legval(g, NL.legder(cR))  # g_R'(xi_a)
    dgL = -NL.legval(-g, NL.legder(cR))  # d/dxi g_R(-xi)
    M3 = np.zeros((ref.Nu, ref.Nf))
    for d in range(nd):
        others = [dd for dd in range(nd) if dd != d]
        for s in range(2):
            for idx in range(ref.nfp):
                sig = (2 * d + s) * ref.nfp + idx
                fidx = [(idx // n ** m) % n for m in range(nd - 1)]
                for rho in range(ref.Nu):
                    ridx = [(rho // n ** dd) % n for dd in range(nd)]
                    if all(ridx[dd] == fidx[m] for m, dd in enumerate(others)):
                        # outward-normal convention: n.g = 1 at own flux point
                        M3[rho, sig] = dgR[ridx[d]] if s == 1 else -dgL[ridx[d]]
    assert np.allclose(np.asarray(ops.M3, float), M3, atol=1e-13)


@pytest.mark.parametrize("etype,p", ETYPES)
def test_fused_equals_unfused(etype, p):
    """Eq 42 (:753-756) and Eq 44 (:772-773): fused operator forms equal the literal forms."""
    ref = RefElement(etype, p)
    o = Operators(ref)
    rng = np.random.default_rng(0)
    u = rng.standard_normal(ref.Nu).astype(LD)
    C = rng.standard_normal(ref.Nf).astype(LD)
    F = rng.standard_normal(ref.nd * ref.Nu).astype(LD)
    D = rng.standard_normal(ref.Nf).astype(LD)
    a = o.M6 @ (C - o.M0 @ u) + o.M4 @ u
    b = o.M6 @ C + (o.M4 - o.M6 @ o.M0) @ u
    assert np.max(np.abs(a - b)) < 1e-15 * max(1, np.max(np.abs(o.M6)) * ref.Nf)
    a = o.M3 @ (D - o.M2 @ F) + o.M1 @ F
    b = o.M3 @ D + (o.M1 - o.M3 @ o.M2) @ F
    assert np.max(np.abs(a - b)) < 1e-15 * max(1, np.max(np.abs(o.M3)) * ref.Nf)
    assert o.M5.shape == (ref.nd * ref.Nf, ref.nd * ref.Nu)
    assert np.array_equal(o.M5[ref.Nf : 2 * ref.Nf, ref.Nu : 2 * ref.Nu], o.M0)
    assert np.all(o.M5[: ref.Nf, ref.Nu :] == 0)


@pytest.mark.parametrize("etype,p", ETYPES)
def test_M6_single_element_gradient_with_exact_trace(etype, p):
    """Eq 9 (:202) with reading A1: if C is the trace of a degree-(p+1)... no: of ANY smooth function
    w whose interpolant is u, then M6 (C - M0 u) + M4 u is the L2 projection-type corrected gradient;
    for w polynomial of degree <= p the jump vanishes and the gradient is exact; for the one-sided
    choice C = w + c (constant shift c on all faces) the correction must be zero-mean-consistent:
    integral of the corrected gradient = boundary integral of C n (Gauss theorem), which pins the
    n (x) M3 structure of M6, its sign and its index roles."""
    ref = RefElement(etype, p)
    o = Operators(ref)
    rng = np.random.default_rng(1)
    u = rng.standard_normal(ref.Nu).astype(LD)
    C = rng.standard_normal(ref.Nf).astype(LD)
    qt = (o.M6 @ (C - o.M0 @ u) + o.M4 @ u).reshape(ref.nd, ref.Nu)
    for d in range(ref.nd):
        lhs = ref.wu @ qt[d]  # integral of q_d over the element
        rhs = np.sum(ref.wf * ref.nf[:, d] * C)  # boundary integral of C n_d
        assert abs(float(lhs - rhs)) < 1e-13


@pytest.mark.parametrize("etype,p", [("tri", 1), ("tri", 2), ("tri", 3), ("tri", 4), ("quad", 3)])
def test_M3_is_the_DG_lifting_weak_form(etype, p):
    """What tells the DG correction from every other admissible one (reading A5; VERDICT r1 soft spot i): the divergence of the
    correction field of flux point sigma, h_sigma = sum_rho M3[rho, sigma] l_rho, is the L2 representer of the weighted point
    evaluation on the face:  int_Omega phi h_sigma = w_sigma phi(x_sigma)  for EVERY phi of degree <= p (an SD- or HU-like
    correction satisfies it for degree <= p - 1 only).  Checked with the test's own quadrature (numpy Gauss-Legendre, Duffy
    map on the triangle) against all monomials -- the strong-form DG equivalence M3 D~ + (M1 - M3 M2) F~ follows from it by
    integration by parts (Eq 8)."""
    from numpy.polynomial.legendre import leggauss

    ref = RefElement(etype, p)
    M3 = np.asarray(Operators(ref).M3, dtype=np.float64)
    g, w = leggauss(p + 4)
    a, b = np.meshgrid(g, g, indexing="ij")
    wa, wb = np.meshgrid(w, w, indexing="ij")
    if etype == "tri":
        xq = np.stack([((1 + a) * (1 - b) / 2 - 1).ravel(), b.ravel()], -1)
        wq = (wa * wb * (1 - b) / 2).ravel()
    else:
        xq, wq = np.stack([a.ravel(), b.ravel()], -1), (wa * wb).ravel()
    Lq = np.asarray(ref.basis(xq)[0], dtype=np.float64)          # l_rho at the quadrature points
    h = Lq @ M3                                                   # h_sigma at the quadrature points
    xf, wf = np.asarray(ref.xf, float), np.asarray(ref.wf, float)
    worst_p, worst_p1 = 0.0, 0.0
    for ea in range(p + 2):
        for eb in range(p + 2 - ea):
            phi_q, phi_f = xq[:, 0] ** ea * xq[:, 1] ** eb, xf[:, 0] ** ea * xf[:, 1] ** eb
            res = np.max(np.abs((wq * phi_q) @ h - wf * phi_f))
            if ea + eb <= p:
                worst_p = max(worst_p, res)
            elif etype == "tri":
                worst_p1 = max(worst_p1, res)
    assert worst_p < 1e-12, worst_p
    if etype == "tri":
        assert worst_p1 > 1e-3  # and not beyond degree p: the identity is sharp
