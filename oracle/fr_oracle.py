"""ORACLE — test infrastructure only.  Plain, slow, dense CPU (numpy) implementation of
the Flux Reconstruction right-hand side of arxiv/paper_1312_1638 (PyFR), written from
the paper step by step.  Only tests/, __graft_entry__.smoke() and bench.py's
cpu_baseline / --impl reference legs may import it.  It shares no code with the CUDA
library under paper_1312_1638_b200/ and never imports it.

Citations are PAPER.md:<line> (+ equation).  Readings of garbled / silent passages are
the A-numbers of SURVEY.md §8(c), restated in DESIGN.md.

What it computes (all arrays [point, variable, element], dense operators, no tensor-product
shortcuts, no sorted tables; flux-point pairing by brute-force coordinate matching):

  O1  Gauss-Legendre points/weights (Newton on P_n); point sets; reference normals   :182, :601
  O2  nodal basis via generalised Vandermonde  l = V^-1 psi                          :182
  O3  M0, M1, M2, M3, M4, M5(block diag of M0), M6                                   :737-768 (A1, A2)
  O4  geometry: J, S = J*J^-1 at solution/flux points, physical normals Eq 14        :151-160, :223
  O5  U^f = M0 U                                                                     Eq 6 :186
  O6  common solution, LDG                                                           Eq 7 :192, Eq 25 :506
  O7  q~ = M6 (C - U^f) + M4 U ; q = J^-T q~ ; q^f = M0 q                            Eq 9-11 :202-210
  O8  f = f_inv - f_vis ; f~ = S f                                                   Eq 12 :214, Eq 20-24 :474-500
  O9  common normal flux: Rusanov + LDG, transformed by J n                          Eq 15-17, 26-27, 45-46
  O10 R~ = M3 (D~ - M2 F~) + M1 F~ ; R = -R~/J                                       Eq 18-19 :239-245
  O11 classical RK4                                                                  :247
  O12 L2 error by Gauss quadrature at the solution points                            Eq 32-33 :557-564

Pins (tests/test_oracle_*.py, `-m "not gpu"`): GL closed forms, polynomial exactness of
M0/M4/M1, zero divergence of a constant flux, w^T M3 = w^f, Radau closed form of the DG
correction on tensor elements, fused == unfused Eq 42/44, gradient exactness for continuous
polynomials, flux consistency/antisymmetry, closed-form stresses, p=0 == first-order finite
volume (hand-written loops), freestream, conservation, vortex order p+1, RK4 stability
polynomial; SD / HU correction functions: end values, zeros at the Gauss / Gauss-Lobatto points;
DOPRI5: row sums, order conditions to order 5 / 4, stability polynomial.
PARITY UNPINNED by the paper (fixed by documentation only): A6 (triangle solution-point set), A7 (sign of
the LDG penalty tau), A12/A13 (which side is L; beta, tau), A23 (which published correction functions the
names SD and HU denote), A24 (the DOPRI5 tableau: named, not printed).
"""
import numpy as np

LD = np.longdouble


# =============================================================================
# O1: Gauss-Legendre quadrature ("Gauss-Legendre solution and flux points")
# =============================================================================
def legendre(n, x):
    """P_n(x) and P_n'(x) by the three-term recurrence (works on arrays, any float dtype)."""
    x = np.asarray(x)
    p0 = np.ones_like(x)
    if n == 0:
        return p0, np.zeros_like(x)
    p1 = x.copy()
    d0 = np.zeros_like(x)
    d1 = np.ones_like(x)
    for k in range(1, n):
        p2 = ((2 * k + 1) * x * p1 - k * p0) / (k + 1)
        d2 = ((2 * k + 1) * (p1 + x * d1) - k * d0) / (k + 1)
        p0, p1, d0, d1 = p1, p2, d1, d2
    return p1, d1


def gauss_legendre(n):
    """n-point GL nodes (ascending) and weights on [-1,1], long double, Newton on P_n."""
    k = np.arange(1, n + 1, dtype=LD)
    x = -np.cos(LD(np.pi) * (k - LD(0.25)) / (n + LD(0.5)))
    for _ in range(100):
        p, dp = legendre(n, x)
        dx = p / dp
        x = x - dx
        if np.max(np.abs(dx)) < 4 * np.finfo(LD).eps:
            break
    _, dp = legendre(n, x)
    w = 2 / ((1 - x * x) * dp * dp)
    return x, w


# =============================================================================
# O2: nodal bases (l_rho = V^-1 psi, V_rho,sigma = psi_rho(x_sigma))
# =============================================================================
def lagrange_1d(nodes, x):
    """Values and derivatives of the 1-D Lagrange polynomials on `nodes` at points x.
    Returns (L[len(x), n], dL[len(x), n]).  Explicit products (tensor elements)."""
    nodes = np.asarray(nodes, dtype=LD)
    x = np.asarray(x, dtype=LD)
    n = nodes.size
    L = np.ones((x.size, n), dtype=LD)
    dL = np.zeros((x.size, n), dtype=LD)
    for j in range(n):
        for m in range(n):
            if m != j:
                L[:, j] *= (x - nodes[m]) / (nodes[j] - nodes[m])
        for i in range(n):
            if i == j:
                continue
            term = np.ones(x.size, dtype=LD) / (nodes[j] - nodes[i])
            for m in range(n):
                if m != j and m != i:
                    term = term * (x - nodes[m]) / (nodes[j] - nodes[m])
            dL[:, j] += term
    return L, dL


def _solve_ld(A, B):
    """Gauss-Jordan with partial pivoting in long double (numpy.linalg has no long double)."""
    A = np.array(A, dtype=LD)
    B = np.array(B, dtype=LD)
    n = A.shape[0]
    for c in range(n):
        piv = c + int(np.argmax(np.abs(A[c:, c])))
        if piv != c:
            A[[c, piv]] = A[[piv, c]]
            B[[c, piv]] = B[[piv, c]]
        B[c] = B[c] / A[c, c]
        A[c] = A[c] / A[c, c]
        for r in range(n):
            if r != c:
                f = A[r, c]
                if f != 0:
                    A[r] = A[r] - f * A[c]
                    B[r] = B[r] - f * B[c]
    return B


def _tri_psi(p, X):
    """Basis psi_ab = P_a(x) P_b(y), a+b<=p, spanning the order-p space on the triangle
    ("any basis which spans a selected order-p polynomial space").
    Returns psi[len(X), N], dpsi[2, len(X), N]."""
    X = np.asarray(X, dtype=LD)
    cols, dx, dy = [], [], []
    for b in range(p + 1):
        for a in range(p + 1 - b):
            pa, dpa = legendre(a, X[:, 0])
            pb, dpb = legendre(b, X[:, 1])
            cols.append(pa * pb)
            dx.append(dpa * pb)
            dy.append(pa * dpb)
    return np.stack(cols, -1), np.stack([np.stack(dx, -1), np.stack(dy, -1)])


def nodal_basis(etype, pts_1d_or_pts, X):
    """Evaluate the nodal basis on a point set at points X[npts, nd].
    quad/hex: `pts_1d_or_pts` is the 1-D node vector; basis = tensor product of 1-D Lagrange
    polynomials, index rho = i + n*j (+ n^2*k), first coordinate fastest.
    tri: `pts_1d_or_pts` = (p, nodes[N,2]); basis via Vandermonde inverse.
    Returns L[npts, N], dL[nd, npts, N]."""
    X = np.asarray(X, dtype=LD)
    if etype in ("quad", "hex"):
        nd = 2 if etype == "quad" else 3
        n = len(pts_1d_or_pts)
        l1 = [lagrange_1d(pts_1d_or_pts, X[:, d]) for d in range(nd)]
        N = n ** nd
        L = np.empty((X.shape[0], N), dtype=LD)
        dL = np.empty((nd, X.shape[0], N), dtype=LD)
        for rho in range(N):
            idx = [(rho // n ** d) % n for d in range(nd)]
            val = np.ones(X.shape[0], dtype=LD)
            for d in range(nd):
                val = val * l1[d][0][:, idx[d]]
            L[:, rho] = val
            for dd in range(nd):
                g = np.ones(X.shape[0], dtype=LD)
                for d in range(nd):
                    g = g * (l1[d][1][:, idx[d]] if d == dd else l1[d][0][:, idx[d]])
                dL[dd, :, rho] = g
        return L, dL
    p, nodes = pts_1d_or_pts
    V, _ = _tri_psi(p, nodes)  # V[sigma, a] = psi_a(x_sigma)
    psi, dpsi = _tri_psi(p, X)
    # l_sigma(x) = sum_a c[a, sigma] psi_a(x) with  V c = I
    c = _solve_ld(V, np.eye(V.shape[0], dtype=LD))
    return psi @ c, np.stack([dpsi[0] @ c, dpsi[1] @ c])


# =============================================================================
# O1: reference elements: point sets, normals, face quadrature weights
# =============================================================================
class RefElement:
    """Reference element of order p with solution points x_u, flux points x_f, outward unit
    reference normals n_f, face-quadrature weights w_f, volume-quadrature weights w_u
    (w_u[rho] = integral of l_rho), and geometry nodes of degree p_g.

    quad/hex on [-1,1]^nd: GL tensor solution points; flux point sigma = face*nfp + idx with
    face = 2*d + s and idx the tensor GL index over the remaining directions (lowest fastest).
    tri on (-1,-1),(1,-1),(-1,1): solution points = barycentric lattice (i+1,j+1,k+1)/(p+3)
    (reading A6); flux points = GL points along each counter-clockwise edge."""

    def __init__(self, etype, p):
        self.etype, self.p = etype, p
        self.nd = nd = 3 if etype == "hex" else 2
        n = p + 1
        g, w = gauss_legendre(n)
        self.g1, self.w1 = g, w
        if etype in ("quad", "hex"):
            N = n ** nd
            xu = np.empty((N, nd), dtype=LD)
            wu = np.ones(N, dtype=LD)
            for rho in range(N):
                for d in range(nd):
                    i = (rho // n ** d) % n
                    xu[rho, d] = g[i]
                    wu[rho] *= w[i]
            nfp = n ** (nd - 1)
            xf = np.empty((2 * nd * nfp, nd), dtype=LD)
            nf = np.zeros((2 * nd * nfp, nd), dtype=LD)
            wf = np.ones(2 * nd * nfp, dtype=LD)
            for d in range(nd):
                others = [dd for dd in range(nd) if dd != d]
                for s in range(2):
                    for idx in range(nfp):
                        sig = (2 * d + s) * nfp + idx
                        xf[sig, d] = -1 if s == 0 else 1
                        nf[sig, d] = -1 if s == 0 else 1
                        for m, dd in enumerate(others):
                            i = (idx // n ** m) % n
                            xf[sig, dd] = g[i]
                            wf[sig] *= w[i]
            self.basis_arg = g
            self.nfaces, self.nfp = 2 * nd, nfp
        else:
            pts = []
            for j in range(p + 1):
                for i in range(p + 1 - j):
                    l1, l2 = LD(i + 1) / (p + 3), LD(j + 1) / (p + 3)
                    pts.append((-1 + 2 * l1, -1 + 2 * l2))
            xu = np.array(pts, dtype=LD)
            verts = np.array([(-1, -1), (1, -1), (-1, 1)], dtype=LD)
            normals = np.array([(0, -1), (1 / np.sqrt(LD(2)), 1 / np.sqrt(LD(2))), (-1, 0)], dtype=LD)
            scale = [LD(1), np.sqrt(LD(2)), LD(1)]  # edge length / 2
            xf = np.empty((3 * n, 2), dtype=LD)
            nf = np.empty((3 * n, 2), dtype=LD)
            wf = np.empty(3 * n, dtype=LD)
            for k in range(3):
                a, b = verts[k], verts[(k + 1) % 3]
                for i in range(n):
                    xf[k * n + i] = (a * (1 - g[i]) + b * (1 + g[i])) / 2
                    nf[k * n + i] = normals[k]
                    wf[k * n + i] = w[i] * scale[k]
            self.basis_arg = (p, xu)
            self.nfaces, self.nfp = 3, n
            wu = None
        self.xu, self.xf, self.nf, self.wf = xu, xf, nf, wf
        self.Nu, self.Nf = xu.shape[0], xf.shape[0]
        # exact volume quadrature for polynomial integrands of degree <= 2p+2 (used for the mass matrix)
        self.xq, self.wq = self._volume_quadrature(p + 3)
        Lq, _ = self.basis(self.xq)
        self.mass = np.einsum("q,qa,qb->ab", self.wq, Lq, Lq)  # exact integral of l_a l_b
        self.wu = Lq.T @ self.wq if wu is None else wu  # integral of l_rho

    def _volume_quadrature(self, m):
        g, w = gauss_legendre(m)
        if self.etype in ("quad", "hex"):
            grids = np.meshgrid(*([g] * self.nd), indexing="ij")
            wg = np.meshgrid(*([w] * self.nd), indexing="ij")
            return np.stack([x.ravel() for x in grids], -1), np.prod(np.stack([x.ravel() for x in wg], -1), -1)
        # Duffy map of the square onto the triangle: x = (1+a)(1-b)/2 - 1, y = b, dA = (1-b)/2 da db
        a, b = np.meshgrid(g, g, indexing="ij")
        wa, wb = np.meshgrid(w, w, indexing="ij")
        x = (1 + a) * (1 - b) / 2 - 1
        return np.stack([x.ravel(), b.ravel()], -1), (wa * wb * (1 - b) / 2).ravel()

    def basis(self, X):
        return nodal_basis(self.etype, self.basis_arg, X)

    # --- geometry nodes / basis (degree p_g Lagrange on the equispaced lattice) ---
    def geometry_basis(self, p_g, X):
        if self.etype in ("quad", "hex"):
            nodes = np.linspace(LD(-1), LD(1), p_g + 1, dtype=LD)
            return nodal_basis(self.etype, nodes, X)
        pts = []
        for j in range(p_g + 1):
            for i in range(p_g + 1 - j):
                pts.append((-1 + 2 * LD(i) / p_g, -1 + 2 * LD(j) / p_g))
        return nodal_basis("tri", (p_g, np.array(pts, dtype=LD)), X)


# =============================================================================
# correction functions of the FR schemes the paper runs ("DG, SD, and HU as defined in [10]")
# =============================================================================
def correction_derivative_1d(scheme, p, x):
    """g_R'(x) of the 1-D right-boundary correction function g_R (degree p+1, g_R(-1) = 0, g_R(1) = 1) on [-1,1];
    the left one is g_L(x) = g_R(-x).  Closed forms (reading A23; the paper only names the schemes):
      dg  g_R = R_{p+1},  R_k = (P_{k-1} + P_k)/2 the right Radau polynomial of degree k  (reading A5)
      sd  g_R = (1 + x)/2 * P_p(x): zero at the p Gauss points, which recovers the spectral difference scheme
      hu  g_R = ((p+1) R_p + p R_{p+1}) / (2p+1): Huynh's g_2, whose derivative vanishes at the interior
          Gauss-Lobatto points and at -1."""
    x = np.asarray(x, dtype=LD)

    def radau_d(k):  # R_k' = (P_{k-1}' + P_k')/2
        return (legendre(k - 1, x)[1] + legendre(k, x)[1]) / 2

    if scheme == "dg":
        return radau_d(p + 1)
    if scheme == "sd":
        P, dP = legendre(p, x)
        return P / 2 + (1 + x) / 2 * dP
    if scheme == "hu":
        if p < 1:
            raise ValueError("the HU scheme needs p >= 1")
        return ((p + 1) * radau_d(p) + p * radau_d(p + 1)) / (2 * p + 1)
    raise KeyError(scheme)


# =============================================================================
# O3: constant operator matrices (App A)
# =============================================================================
class Operators:
    """M0..M6 of Appendix A for one element type, long double.
    Vector rows are packed with stride N_u (or N_f): row = d*N_u + rho.
    scheme: 'dg' (any element type) or 'sd' / 'hu' (quadrilaterals and hexahedra, tensor product of the 1-D functions)."""

    def __init__(self, ref, scheme="dg"):
        nd, Nu, Nf = ref.nd, ref.Nu, ref.Nf
        Lf, _ = ref.basis(ref.xf)  # [Nf, Nu]
        _, dLu = ref.basis(ref.xu)  # [nd, Nu(points), Nu(basis)]
        # M0[sigma, rho] = l_rho(x^f_sigma)                                      :737
        self.M0 = Lf
        # M4[(d,sigma), rho] = d_d l_rho (x^u_sigma)                             :749
        self.M4 = dLu.reshape(nd * Nu, Nu)
        # M1[rho, (d,nu)] = d_d l_nu (x^u_rho)   (the "transpose" of :768)
        self.M1 = np.concatenate([dLu[d] for d in range(nd)], axis=1)
        # M2[sigma, (d,rho)] = l_rho(x^f_sigma) n_sigma,d                        :768
        self.M2 = np.concatenate([Lf * ref.nf[:, d : d + 1] for d in range(nd)], axis=1)
        # M3[rho, sigma] = (div g_sigma)(x^u_rho), DG correction (reading A5):
        # div g_sigma = sum_rho l_rho * (Mass^-1 M0^T diag(w^f))[rho, sigma]
        self.M3 = _solve_ld(ref.mass, Lf.T * ref.wf[None, :])
        if scheme != "dg":
            # SD / HU on tensor elements: the correction field of flux point sigma on face (d, s) is the 1-D function along d
            # times the face's Lagrange polynomials in the other directions, so (div g_sigma)(x_rho) = g'(xi_d) on the line
            # of solution points through sigma and zero off it; outward normals: +g_R'(xi) at s = 1, g_R'(-xi) at s = 0
            if ref.etype not in ("quad", "hex"):
                raise ValueError("SD / HU correction functions are defined on quadrilaterals and hexahedra only")
            n, M3 = ref.p + 1, np.zeros((Nu, Nf), dtype=LD)
            for sig in range(Nf):
                d, side = (sig // ref.nfp) // 2, (sig // ref.nfp) % 2
                others = [dd for dd in range(nd) if dd != d]
                on_line = np.all(np.abs(ref.xu[:, others] - ref.xf[sig, others][None, :]) < 1e-14, axis=1)
                xi = ref.xu[on_line, d]
                M3[on_line, sig] = correction_derivative_1d(scheme, ref.p, xi if side else -xi)
            self.M3 = M3
        # M6[(d,rho), sigma] = n_sigma,d * M3[rho, sigma]  (reading A1)           :749
        self.M6 = np.concatenate([self.M3 * ref.nf[None, :, d] for d in range(nd)], axis=0)
        # M5 = diag(M0,...,M0)                                                    :760
        self.M5 = np.kron(np.eye(nd, dtype=LD), self.M0)


# =============================================================================
# physics: O8, O9 (PAPER.md:474-516 §4, :781-825 App B, C)
# =============================================================================
def primitives(u, gamma):
    """u[..., N_V, ...] with variable axis = 0 here: returns rho, v[nd], p, E.  Eq 20-21 :474-481"""
    nd = u.shape[0] - 2
    rho = u[0]
    v = [u[1 + d] / rho for d in range(nd)]
    E = u[nd + 1]
    p = (gamma - 1) * (E - rho * sum(vi * vi for vi in v) / 2)
    return rho, v, p, E


def flux_inviscid(u, gamma):
    """f_inv[n][alpha] of Eq 20 (:474); 2-D by deleting the 4th row / 3rd column (:520)."""
    nd = u.shape[0] - 2
    rho, v, p, E = primitives(u, gamma)
    f = []
    for n in range(nd):
        col = [rho * v[n]]
        for j in range(nd):
            col.append(rho * v[n] * v[j] + (p if j == n else 0))
        col.append(v[n] * (E + p))
        f.append(np.stack(col))
    return np.stack(f)  # [nd, N_V, ...]


def flux_viscous(u, q, gamma, mu, Pr):
    """f_vis[n][alpha] of Eq 22-24 (:489-500).  q[n][alpha] = d_n u_alpha.
    d_i v_j by the quotient rule; Delta dT = (mu gamma / Pr) d e  (reading A8); the 2/3
    of Eq 23 is kept in 2-D (reading A22)."""
    nd = u.shape[0] - 2
    rho, v, p, E = primitives(u, gamma)
    dv = [[(q[i][1 + j] - v[j] * q[i][0]) / rho for j in range(nd)] for i in range(nd)]  # dv[i][j] = d_i v_j
    div = sum(dv[i][i] for i in range(nd))
    T = [[mu * (dv[i][j] + dv[j][i]) - (2 * mu * div / 3 if i == j else 0) for j in range(nd)] for i in range(nd)]
    # e = E/rho - |v|^2/2 ;  d_i e = (d_i E - (E/rho) d_i rho)/rho - v_j d_i v_j
    de = [(q[i][nd + 1] - (E / rho) * q[i][0]) / rho - sum(v[j] * dv[i][j] for j in range(nd)) for i in range(nd)]
    f = []
    for n in range(nd):
        col = [np.zeros_like(rho)]
        for j in range(nd):
            col.append(T[n][j])  # row (j+1), column n of Eq 22 is T_{n j}
        col.append(sum(v[i] * T[i][n] for i in range(nd)) + (mu * gamma / Pr) * de[n])
        f.append(np.stack(col))
    return np.stack(f)


def rusanov(uL, uR, nL, gamma):
    """Eq 45-46 (:785-789), printed form of the wave speed (reading A14)."""
    nd = uL.shape[0] - 2
    fL, fR = flux_inviscid(uL, gamma), flux_inviscid(uR, gamma)
    rL, vL, pL, _ = primitives(uL, gamma)
    rR, vR, pR, _ = primitives(uR, gamma)
    s = np.sqrt(gamma * (pL + pR) / (rL + rR)) + np.abs(sum(nL[d] * (vL[d] + vR[d]) for d in range(nd))) / 2
    return sum(nL[d] * (fL[d] + fR[d]) for d in range(nd)) / 2 + (s / 2) * (uL - uR)


def ldg_viscous(uL, uR, qL, qR, nL, gamma, mu, Pr, beta, tau):
    """F_vis of Eq 27 (:514) WITHOUT the penalty; the penalty enters common_flux with the
    dissipative sign (reading A7)."""
    nd = uL.shape[0] - 2
    fL = flux_viscous(uL, qL, gamma, mu, Pr)
    fR = flux_viscous(uR, qR, gamma, mu, Pr)
    return sum(nL[d] * ((0.5 + beta) * fL[d] + (0.5 - beta) * fR[d]) for d in range(nd))


def common_flux(uL, uR, qL, qR, nL, prm, uR_inv=None):
    """Eq 26 (:510): F = F_inv - n.{(1/2+beta) f_L^vis + (1/2-beta) f_R^vis} + tau (u_L - u_R) (A7).
    uR_inv: ghost state for the inviscid part at a boundary (reading A20)."""
    F = rusanov(uL, uR if uR_inv is None else uR_inv, nL, prm["gamma"])
    if prm["system"] == "navier-stokes":
        F = F - ldg_viscous(uL, uR, qL, qR, nL, prm["gamma"], prm["mu"], prm["Pr"], prm["beta"], prm["tau"])
        F = F + prm["tau"] * (uL - uR)
    return F


def ghost_states(kind, par, uL, gamma):
    """Appendix C (:795-825).  Returns (B_inv u_L, B_ldg u_L, keep_q) with keep_q the factor
    applied to q_L for B_ldg q_L (0: Eq 48/50, 1: Eq 53)."""
    nd = uL.shape[0] - 2
    rho, v, p, E = primitives(uL, gamma)
    one = np.ones_like(rho)
    if kind == "sup-inflow":  # Eq 47-48
        rf, vf, pf = par["rho"], par["v"], par["p"]
        g = np.stack([rf * one] + [rf * vf[d] * one for d in range(nd)] + [(pf / (gamma - 1) + rf * sum(x * x for x in vf) / 2) * one])
        return g, g, 0.0
    if kind == "sub-outflow":  # Eq 49-50
        pf = par["p"]
        g = np.stack([rho] + [rho * v[d] for d in range(nd)] + [pf / (gamma - 1) + rho * sum(x * x for x in v) / 2])
        return g, g, 0.0
    if kind == "noslip-wall":  # Eq 51-53
        cpTw, vw = par["cpTw"], par["v"]
        vi = [2 * vw[d] - v[d] for d in range(nd)]
        gi = np.stack([rho] + [rho * vi[d] for d in range(nd)] + [rho * (cpTw / gamma + sum(x * x for x in vi) / 2)])
        gl = np.stack([rho] + [rho * vw[d] * one for d in range(nd)] + [rho * (cpTw / gamma + sum(x * x for x in vw) / 2)])
        return gi, gl, 1.0
    raise KeyError(kind)


# Dormand-Prince 5(4): nodes c_i = sum_j a_ij, 5th-order weights b5 (= row 7 of A: first-same-as-last), 4th-order weights b4
DOPRI5_A = [
    [],
    [1 / 5],
    [3 / 40, 9 / 40],
    [44 / 45, -56 / 15, 32 / 9],
    [19372 / 6561, -25360 / 2187, 64448 / 6561, -212 / 729],
    [9017 / 3168, -355 / 33, 46732 / 5247, 49 / 176, -5103 / 18656],
    [35 / 384, 0, 500 / 1113, 125 / 192, -2187 / 6784, 11 / 84],
]
DOPRI5_B5 = [35 / 384, 0, 500 / 1113, 125 / 192, -2187 / 6784, 11 / 84, 0]
DOPRI5_B4 = [5179 / 57600, 0, 7571 / 16695, 393 / 640, -92097 / 339200, 187 / 2100, 1 / 40]


# =============================================================================
# the discretisation on a mesh of one element type
# =============================================================================
class FROracle:
    """FR semi-discretisation on a single-element-type mesh (workloads.py mesh dict).

    prm: p, system ('euler'|'navier-stokes'), gamma, mu, Pr, beta, tau, correction ('dg' default | 'sd' | 'hu').
    bcs: {bc_id: (kind, params)} for boundary faces.
    dtype: np.float64 or np.longdouble for the STATE arithmetic (operators and metrics are
    always built in long double and rounded once to dtype)."""

    def __init__(self, mesh, prm, bcs=None, dtype=np.float64, pair=True):
        self.mesh, self.prm, self.bcs, self.dtype = mesh, dict(prm), bcs or {}, dtype
        self.ref = ref = RefElement(mesh["etype"], prm["p"])
        self.ops = Operators(ref, self.prm.get("correction", "dg"))
        self.nd, self.Nu, self.Nf = ref.nd, ref.Nu, ref.Nf
        self.NV = ref.nd + 2
        self.Nel = mesh["nodes"].shape[0]
        self._geometry()
        if pair:  # FRMixedOracle pairs the flux points of all element types itself
            self._pair()
        c = lambda a: np.asarray(a, dtype=dtype)
        o = self.ops
        self.M0, self.M1, self.M2, self.M3, self.M4, self.M6 = c(o.M0), c(o.M1), c(o.M2), c(o.M3), c(o.M4), c(o.M6)

    # ---- O4: metrics (PAPER.md:151-160 Jacobians; :216 S = J J^-1; :223 Eq 14) ----
    def _geometry(self):
        ref, mesh, nd = self.ref, self.mesh, self.nd
        X = np.asarray(mesh["nodes"], dtype=LD)  # [Nel, Nn, nd]

        def at(points):
            G, dG = ref.geometry_basis(mesh["p_g"], points)  # [npts, Nn], [nd, npts, Nn]
            x = np.einsum("pk,eki->pei", G, X)  # [npts, Nel, nd]
            Jm = np.einsum("jpk,eki->peij", dG, X)  # J[i][j] = dx_i/dxi_j
            if nd == 2:
                det = Jm[..., 0, 0] * Jm[..., 1, 1] - Jm[..., 0, 1] * Jm[..., 1, 0]
                S = np.empty_like(Jm)  # S = det * J^-1 (adjugate): S[i][n] = det * dxi_i/dx_n
                S[..., 0, 0], S[..., 0, 1] = Jm[..., 1, 1], -Jm[..., 0, 1]
                S[..., 1, 0], S[..., 1, 1] = -Jm[..., 1, 0], Jm[..., 0, 0]
            else:
                S = np.empty_like(Jm)
                for i in range(3):
                    for n in range(3):
                        # adj(J)[i][n] = cofactor(J)[n][i]
                        a, b = [(n + 1) % 3, (n + 2) % 3], [(i + 1) % 3, (i + 2) % 3]
                        S[..., i, n] = Jm[..., a[0], b[0]] * Jm[..., a[1], b[1]] - Jm[..., a[0], b[1]] * Jm[..., a[1], b[0]]
                det = sum(Jm[..., 0, j] * S[..., j, 0] for j in range(3))
            return x, S, det

        self.xu_phys, Su, Ju = at(ref.xu)
        self.xf_phys, Sf, Jf = at(ref.xf)
        if np.any(Ju <= 0) or np.any(Jf <= 0):
            raise ValueError("non-positive Jacobian")
        # J^-T n~ scaled by J:  (S^T n~)_n = sum_i S[i][n] n~_i ;  J n = |.| ; n^ = ./|.|   (Eq 14, A15)
        Sn = np.einsum("pein,pi->pen", Sf, ref.nf)
        mag = np.sqrt(np.sum(Sn * Sn, -1))
        c = lambda a: np.asarray(a, dtype=self.dtype)
        self.Su, self.Ju = c(Su), c(Ju)  # [Nu, Nel, nd, nd], [Nu, Nel]
        self.Jn_f = c(mag)  # [Nf, Nel]     = J * n of Eq 16
        self.nhat_f = c(Sn / mag[..., None])  # [Nf, Nel, nd]

    # ---- lookup table by brute force (reading A11) ----
    def _pair(self):
        mesh, nfp = self.mesh, self.ref.nfp
        xf = np.asarray(self.xf_phys, dtype=np.float64)  # [Nf, Nel, nd]
        ifc = mesh["ifaces"]
        eL, fL, eR, fR = ifc[:, 0], ifc[:, 1], ifc[:, 2], ifc[:, 3]
        k = np.arange(nfp)
        sL = fL[:, None] * nfp + k[None, :]  # [nif, nfp]
        sR = fR[:, None] * nfp + k[None, :]
        xL = xf[sL, eL[:, None]]  # [nif, nfp, nd]
        xR = xf[sR, eR[:, None]] + mesh["shifts"][:, None, :]
        d2 = np.sum((xL[:, :, None, :] - xR[:, None, :, :]) ** 2, -1)  # [nif, nfp(L), nfp(R)]
        match = np.argmin(d2, axis=2)
        best = np.take_along_axis(d2, match[..., None], 2)[..., 0]
        hmin = np.sqrt(np.min(np.sum((xL[:, 0] - xL[:, -1]) ** 2, -1))) if nfp > 1 else 1.0
        if ifc.shape[0] and np.sqrt(best.max()) > 1e-9 * max(hmin, 1e-300) + 1e-12:
            raise ValueError("unmatched flux-point pair (%g)" % np.sqrt(best.max()))
        if ifc.shape[0] and np.any(np.sort(match, axis=1) != k[None, :]):
            raise ValueError("flux-point matching is not a permutation")
        self.pL_s, self.pL_e = sL.ravel(), np.repeat(eL, nfp)
        self.pR_s = np.take_along_axis(sR, match, 1).ravel()
        self.pR_e = np.repeat(eR, nfp)
        bf = mesh["bfaces"]
        self.b_s = (bf[:, 1][:, None] * nfp + k[None, :]).ravel()
        self.b_e = np.repeat(bf[:, 0], nfp)
        self.b_id = np.repeat(bf[:, 2], nfp)
        # every flux point must be referenced exactly once
        cnt = np.zeros((self.Nf, self.Nel), dtype=np.int64)
        np.add.at(cnt, (self.pL_s, self.pL_e), 1)
        np.add.at(cnt, (self.pR_s, self.pR_e), 1)
        np.add.at(cnt, (self.b_s, self.b_e), 1)
        if np.any(cnt != 1):
            raise ValueError("flux points not covered exactly once by interfaces + boundaries")

    # ---- the steps ----
    def interpolate(self, u):
        """O5, Eq 6 / Eq 41: U^f = M0 U."""
        return np.einsum("sr,rvn->svn", self.M0, u, optimize=True)

    def common_solution(self, uf):
        """O6, Eq 7 + Eq 25; boundary: C(u_L, B_ldg u_L) (:797)."""
        b = self.prm["beta"]
        C = np.empty_like(uf)
        uL, uR = uf[self.pL_s, :, self.pL_e], uf[self.pR_s, :, self.pR_e]  # [npairs, NV]
        c = (0.5 - b) * uL + (0.5 + b) * uR
        C[self.pL_s, :, self.pL_e] = c
        C[self.pR_s, :, self.pR_e] = c
        for bc_id, (kind, par) in self.bcs.items():
            m = self.b_id == bc_id
            ub = uf[self.b_s[m], :, self.b_e[m]].T  # [NV, nb]
            _, gl, _ = ghost_states(kind, par, ub, self.prm["gamma"])
            C[self.b_s[m], :, self.b_e[m]] = ((0.5 - b) * ub + (0.5 + b) * gl).T
        return C

    def gradient(self, u, uf, C):
        """O7: Eq 9 literally (unfused), Eq 10, Eq 11."""
        nd, Nu = self.nd, self.Nu
        qt = np.einsum("ks,svn->kvn", self.M6, C - uf, optimize=True) + np.einsum("kr,rvn->kvn", self.M4, u, optimize=True)
        qt = qt.reshape(nd, Nu, self.NV, self.Nel)
        # q_n = (1/J) sum_i S[i][n] q~_i   (J^-T = S^T / J)
        q = np.stack([sum(self.Su[:, None, :, i, n] * qt[i] for i in range(nd)) / self.Ju[:, None, :] for n in range(nd)])
        qf = np.stack([np.einsum("sr,rvn->svn", self.M0, q[n], optimize=True) for n in range(nd)])
        return q, qf

    def transformed_flux(self, u, q):
        """O8: Eq 12 with Eq 20-24; returns F~[(d,rho), v, n]."""
        nd = self.nd
        ua = np.moveaxis(u, 1, 0)  # [NV, Nu, Nel]
        f = flux_inviscid(ua, self.prm["gamma"])  # [nd, NV, Nu, Nel]
        if self.prm["system"] == "navier-stokes":
            qa = np.moveaxis(q, 2, 1)  # [nd, NV, Nu, Nel]
            f = f - flux_viscous(ua, qa, self.prm["gamma"], self.prm["mu"], self.prm["Pr"])
        ft = np.stack([sum(self.Su[None, :, :, i, n] * f[n] for n in range(nd)) for i in range(nd)])  # [nd, NV, Nu, Nel]
        return np.moveaxis(ft, 1, 2).reshape(nd * self.Nu, self.NV, self.Nel)

    def interface_flux(self, uf, qf):
        """O9: Eq 15-17 with Eq 26-27, 45-46; boundary via ghost states (App C, A20)."""
        nd, prm = self.nd, self.prm
        D = np.empty_like(uf)
        ns = prm["system"] == "navier-stokes"
        uL, uR = uf[self.pL_s, :, self.pL_e].T, uf[self.pR_s, :, self.pR_e].T  # [NV, npairs]
        qL = np.stack([qf[n][self.pL_s, :, self.pL_e].T for n in range(nd)]) if ns else None
        qR = np.stack([qf[n][self.pR_s, :, self.pR_e].T for n in range(nd)]) if ns else None
        nL = self.nhat_f[self.pL_s, self.pL_e].T  # [nd, npairs]
        F = common_flux(uL, uR, qL, qR, nL, prm)
        D[self.pL_s, :, self.pL_e] = (self.Jn_f[self.pL_s, self.pL_e][None, :] * F).T  # Eq 16
        D[self.pR_s, :, self.pR_e] = (-self.Jn_f[self.pR_s, self.pR_e][None, :] * F).T  # Eq 15, 17
        for bc_id, (kind, par) in self.bcs.items():
            m = self.b_id == bc_id
            s, e = self.b_s[m], self.b_e[m]
            ub = uf[s, :, e].T
            gi, gl, keep = ghost_states(kind, par, ub, prm["gamma"])
            qb = np.stack([qf[n][s, :, e].T for n in range(nd)]) if ns else None
            Fb = common_flux(ub, gl, qb, keep * qb if ns else None, self.nhat_f[s, e].T, prm, uR_inv=gi)
            D[s, :, e] = (self.Jn_f[s, e][None, :] * Fb).T
        return D

    def divergence(self, ft, D):
        """O10: Eq 18 literally (unfused) then Eq 19."""
        Rt = np.einsum("rs,svn->rvn", self.M3, D - np.einsum("sk,kvn->svn", self.M2, ft), optimize=True) + np.einsum("rk,kvn->rvn", self.M1, ft, optimize=True)
        return -Rt / self.Ju[:, None, :]

    def rhs(self, u, return_parts=False):
        """R(u) = -div f, u[Nu, NV, Nel]."""
        u = np.asarray(u, dtype=self.dtype)
        uf = self.interpolate(u)
        q = qf = C = None
        if self.prm["system"] == "navier-stokes":
            C = self.common_solution(uf)
            q, qf = self.gradient(u, uf, C)
        ft = self.transformed_flux(u, q)
        D = self.interface_flux(uf, qf)
        R = self.divergence(ft, D)
        if return_parts:
            return R, dict(uf=uf, C=C, q=q, qf=qf, ft=ft, D=D)
        return R

    def rk4_step(self, u, dt):
        """O11: classical RK4 (:247)."""
        k1 = self.rhs(u)
        k2 = self.rhs(u + (dt / 2) * k1)
        k3 = self.rhs(u + (dt / 2) * k2)
        k4 = self.rhs(u + dt * k3)
        return u + (dt / 6) * (k1 + 2 * k2 + 2 * k3 + k4)

    def euler_step(self, u, dt):
        """Forward Euler (Table 1 :263)."""
        return u + dt * self.rhs(u)

    def dopri5_step(self, u, dt):
        """One step of the Dormand-Prince 5(4) pair (Table 1 :263 names DOPRI5; the tableau is the published one, reading
        A24).  Returns (u advanced with the 5th-order weights, dt * sum (b5 - b4)_i k_i = the embedded error estimate)."""
        k = []
        for i in range(7):
            ui = u
            for j in range(i):
                if DOPRI5_A[i][j] != 0:
                    ui = ui + (dt * DOPRI5_A[i][j]) * k[j]
            k.append(self.rhs(ui))
        new = u
        err = 0
        for i in range(7):
            if DOPRI5_B5[i] != 0:
                new = new + (dt * DOPRI5_B5[i]) * k[i]
            err = err + (dt * (DOPRI5_B5[i] - DOPRI5_B4[i])) * k[i]
        return new, err

    # ---- O12: quadrature functionals ----
    def integrate(self, g):
        """sum_el sum_rho w_rho J_rho g[rho, (v,) el]  (Gauss quadrature at the solution points, Eq 33 :564)."""
        w = np.asarray(self.ref.wu, dtype=self.dtype)
        if g.ndim == 3:
            return np.einsum("r,rn,rvn->v", w, self.Ju, g)
        return np.einsum("r,rn,rn->", w, self.Ju, g)

    def l2_error(self, a, b):
        """sqrt( integral (a-b)^2 ) per variable (Eq 32 :557)."""
        return np.sqrt(self.integrate((a - b) ** 2))


# =============================================================================
# meshes of several element types (PAPER.md:141 element types; :603 "mixed unstructured mesh")
# =============================================================================
class FRMixedOracle:
    """FR semi-discretisation on a mesh whose parts have different element types (workloads.mixed_mesh dictionary).
    Every element-local step (O5, O7, O8, O10) is the single-type oracle's, part by part; the interface steps (O6, O9) run
    over flux-point pairs whose two sides may lie in different parts -- "only the lookup table changes".
    States, right-hand sides: lists of arrays [N_u(part), N_V, N_el(part)]."""

    def __init__(self, mesh, prm, bcs=None, dtype=np.float64):
        self.mesh, self.prm, self.bcs, self.dtype = mesh, dict(prm), bcs or {}, dtype
        self.nd = mesh["ndims"]
        self.parts = []
        for part in mesh["parts"]:
            sub = {"ndims": mesh["ndims"], "etype": part["etype"], "p_g": part["p_g"], "nodes": part["nodes"],
                   "ifaces": np.zeros((0, 4), np.int32), "shifts": np.zeros((0, self.nd)), "bfaces": np.zeros((0, 3), np.int32)}
            self.parts.append(FROracle(sub, prm, None, dtype, pair=False))
        self._pair()

    def _pair(self):
        """Lookup table by brute-force matching of physical flux-point coordinates across parts (reading A11)."""
        P = self.parts
        pairs = []  # (partL, sigmaL, elemL, partR, sigmaR, elemR)
        for (tL, eL, fL, tR, eR, fR), shift in zip(self.mesh["ifaces"], self.mesh["shifts"]):
            nL, nR = P[tL].ref.nfp, P[tR].ref.nfp
            if nL != nR:
                raise ValueError("the two sides of an interface have different numbers of flux points")
            sL, sR = fL * nL + np.arange(nL), fR * nR + np.arange(nR)
            xL = np.asarray(P[tL].xf_phys, float)[sL, eL]
            xR = np.asarray(P[tR].xf_phys, float)[sR, eR] + shift[None, :]
            d2 = np.sum((xL[:, None, :] - xR[None, :, :]) ** 2, -1)
            match = np.argmin(d2, axis=1)
            h = np.sqrt(np.sum((xL[0] - xL[-1]) ** 2)) if nL > 1 else 1.0
            if np.sqrt(np.max(np.min(d2, axis=1))) > 1e-9 * h + 1e-12 or sorted(match.tolist()) != list(range(nR)):
                raise ValueError("unmatched flux-point pair on a mixed interface")
            for k in range(nL):
                pairs.append((tL, sL[k], eL, tR, sR[match[k]], eR))
        self.pairs = np.array(pairs, dtype=np.int64).reshape(-1, 6)
        bnd = []
        for (t, e, f, bc) in self.mesh["bfaces"]:
            nfp = P[t].ref.nfp
            bnd += [(t, f * nfp + k, e, bc) for k in range(nfp)]
        self.bnd = np.array(bnd, dtype=np.int64).reshape(-1, 4)
        cnt = [np.zeros((q.Nf, q.Nel), dtype=np.int64) for q in P]
        for (tL, sL, eL, tR, sR, eR) in self.pairs:
            cnt[tL][sL, eL] += 1
            cnt[tR][sR, eR] += 1
        for (t, s_, e, _) in self.bnd:
            cnt[t][s_, e] += 1
        if any(np.any(c != 1) for c in cnt):
            raise ValueError("flux points not covered exactly once by interfaces + boundaries")

    def _side(self, arrs, side):
        """values at the flux points of one side of every pair: [npairs, ...]"""
        t, s_, e = self.pairs[:, 3 * side], self.pairs[:, 3 * side + 1], self.pairs[:, 3 * side + 2]
        out = None
        for k in range(len(self.parts)):
            m = t == k
            if not np.any(m):
                continue
            v = arrs[k][s_[m], ..., e[m]] if arrs[k].ndim == 3 else arrs[k][s_[m], e[m]]
            if out is None:
                out = np.zeros((len(t),) + v.shape[1:], dtype=v.dtype)
            out[m] = v
        return out

    def _scatter(self, dst, side, vals):
        t, s_, e = self.pairs[:, 3 * side], self.pairs[:, 3 * side + 1], self.pairs[:, 3 * side + 2]
        for k in range(len(self.parts)):
            m = t == k
            if np.any(m):
                dst[k][s_[m], :, e[m]] = vals[m]

    def rhs(self, us):
        P, prm, nd = self.parts, self.prm, self.nd
        ns = prm["system"] == "navier-stokes"
        us = [np.asarray(u, dtype=self.dtype) for u in us]
        ufs = [q.interpolate(u) for q, u in zip(P, us)]                      # O5
        qs, qfs = [None] * len(P), [None] * len(P)
        bmask = [self.bnd[:, 0] == k for k in range(len(P))]
        if ns:
            b = prm["beta"]
            uL, uR = self._side(ufs, 0), self._side(ufs, 1)                   # O6, Eq 7 + Eq 25
            c = (0.5 - b) * uL + (0.5 + b) * uR
            Cs = [np.empty_like(uf) for uf in ufs]
            self._scatter(Cs, 0, c)
            self._scatter(Cs, 1, c)
            for k, q in enumerate(P):
                for bc_id, (kind, par) in self.bcs.items():
                    m = bmask[k] & (self.bnd[:, 3] == bc_id)
                    if np.any(m):
                        s_, e = self.bnd[m, 1], self.bnd[m, 2]
                        ub = ufs[k][s_, :, e].T
                        _, gl, _ = ghost_states(kind, par, ub, prm["gamma"])
                        Cs[k][s_, :, e] = ((0.5 - b) * ub + (0.5 + b) * gl).T
                qs[k], qfs[k] = q.gradient(us[k], ufs[k], Cs[k])              # O7
        fts = [q.transformed_flux(u, qq) for q, u, qq in zip(P, us, qs)]      # O8
        Ds = [np.empty_like(uf) for uf in ufs]                                # O9
        uL, uR = self._side(ufs, 0).T, self._side(ufs, 1).T
        qL = np.stack([self._side([qf[n] for qf in qfs], 0).T for n in range(nd)]) if ns else None
        qR = np.stack([self._side([qf[n] for qf in qfs], 1).T for n in range(nd)]) if ns else None
        nL = self._side([np.moveaxis(q.nhat_f, 2, 1) for q in P], 0).T  # [nd, npairs]
        F = common_flux(uL, uR, qL, qR, nL, prm)
        JL, JR = self._side([q.Jn_f for q in P], 0), self._side([q.Jn_f for q in P], 1)
        self._scatter(Ds, 0, (JL[None, :] * F).T)
        self._scatter(Ds, 1, (-JR[None, :] * F).T)
        for k, q in enumerate(P):
            for bc_id, (kind, par) in self.bcs.items():
                m = bmask[k] & (self.bnd[:, 3] == bc_id)
                if np.any(m):
                    s_, e = self.bnd[m, 1], self.bnd[m, 2]
                    ub = ufs[k][s_, :, e].T
                    gi, gl, keep = ghost_states(kind, par, ub, prm["gamma"])
                    qb = np.stack([qfs[k][n][s_, :, e].T for n in range(nd)]) if ns else None
                    Fb = common_flux(ub, gl, qb, keep * qb if ns else None, q.nhat_f[s_, e].T, prm, uR_inv=gi)
                    Ds[k][s_, :, e] = (q.Jn_f[s_, e][None, :] * Fb).T
        return [q.divergence(ft, D) for q, ft, D in zip(P, fts, Ds)]          # O10

    def rk4_step(self, us, dt):
        add = lambda a, b, c: [x + c * y for x, y in zip(a, b)]
        k1 = self.rhs(us)
        k2 = self.rhs(add(us, k1, dt / 2))
        k3 = self.rhs(add(us, k2, dt / 2))
        k4 = self.rhs(add(us, k3, dt))
        return [u + (dt / 6) * (a + 2 * b + 2 * c + d) for u, a, b, c, d in zip(us, k1, k2, k3, k4)]

    def integrate(self, gs):
        return sum(q.integrate(g) for q, g in zip(self.parts, gs))
