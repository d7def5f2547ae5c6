"""Seeded synthetic inputs shared by the oracle tests, the GPU parity tests and bench.py.

This module holds NO arithmetic of the FR method: it only lays down meshes (node
coordinates + face-level connectivity) and evaluates analytic initial states at
caller-supplied physical coordinates.  The oracle (`oracle/`) and the CUDA
library (`paper_1312_1638_b200/`) both consume its arrays; neither imports the
other.  Recipes are those of SURVEY.md §8(d) / DESIGN.md "Input recipe"; they
stand in for the paper's structured periodic hex workloads (Table 5
mesh, :709 §7 slab) and its unstructured 2-D meshes (:603), which are not
available.

Mesh dictionary (what `fr_setup_mesh` and the oracle take):
  ndims    2 | 3
  etype    'quad' | 'tri' | 'hex'
  p_g      geometry degree
  nodes    float64 [n_elems, n_nodes(p_g), ndims]; tensor lattice, first reference
           coordinate fastest, equispaced on [-1,1]; triangle: lattice rows j=0..p_g,
           i=0..p_g-j on the reference triangle (-1,-1),(1,-1),(-1,1)
  ifaces   int32 [n_if, 4] = (elemL, faceL, elemR, faceR)   (order significant, A12)
  shifts   float64 [n_if, ndims]; x_L(flux point) = x_R(flux point) + shift
  bfaces   int32 [n_b, 3] = (elem, face, bc_id)
Faces: quad/hex face = 2*d + s (d = reference direction, s = 0 at -1, 1 at +1);
triangle face k = edge from vertex k to vertex (k+1)%3, counter-clockwise.
"""
import numpy as np

ETYPE_ND = {"quad": 2, "tri": 2, "hex": 3}


def n_solution_points(etype, p):
    n = p + 1
    return {"quad": n * n, "hex": n ** 3, "tri": n * (n + 1) // 2}[etype]


def n_flux_points(etype, p):
    n = p + 1
    return {"quad": 4 * n, "hex": 6 * n * n, "tri": 3 * n}[etype]


# ----------------------------------------------------------------------------
# structured tensor-product meshes (quad / hex)
# ----------------------------------------------------------------------------
def box_mesh(shape, lengths, p_g=1, periodic=True, warp=None, origin=None):
    """Structured quad (len(shape)==2) or hex (==3) mesh of a box.

    shape    elements per direction, x fastest in the element numbering
    lengths  box side lengths
    periodic bool or per-direction tuple; non-periodic directions produce
             boundary faces with bc_id = 2*d+s
    warp     optional callable X[...,nd] -> displacement[...,nd] added to every
             geometry node (must vanish / be periodic on the box boundary)
    L side of every interior face = element on the low-coordinate side, its +d face;
    on a periodic wrap the element at the high end is L.
    """
    nd = len(shape)
    shape = tuple(int(s) for s in shape)
    lengths = tuple(float(l) for l in lengths)
    origin = (0.0,) * nd if origin is None else tuple(origin)
    if isinstance(periodic, bool):
        periodic = (periodic,) * nd
    m = p_g + 1
    n_el = int(np.prod(shape))
    # element multi-index, x fastest
    eidx = np.stack(np.unravel_index(np.arange(n_el), shape[::-1]), axis=-1)[:, ::-1]  # [n_el, nd] (ix,iy,iz)
    # node lattice multi-index, first coordinate fastest
    nidx = np.stack(np.unravel_index(np.arange(m ** nd), (m,) * nd), axis=-1)[:, ::-1]  # [n_nodes, nd]
    h = np.array(lengths) / np.array(shape)
    # global lattice coordinate in units of h/p_g -> bitwise identical shared nodes
    gl = eidx[:, None, :] * p_g + nidx[None, :, :]
    nodes = np.array(origin)[None, None, :] + gl * (h / p_g)[None, None, :]
    if warp is not None:
        # evaluate the warp at the *periodically reduced* lattice point so that
        # periodic images receive bit-identical displacements
        glr = gl % (np.array(shape) * p_g)[None, None, :]
        base = np.array(origin)[None, None, :] + glr * (h / p_g)[None, None, :]
        nodes = nodes + warp(base)
    ifaces, shifts, bfaces = [], [], []
    strides = [int(np.prod(shape[:d])) for d in range(nd)]
    for d in range(nd):
        idx = eidx[:, d]
        e = np.arange(n_el)
        interior = idx < shape[d] - 1
        eL = e[interior]
        eR = eL + strides[d]
        ifaces.append(np.stack([eL, np.full_like(eL, 2 * d + 1), eR, np.full_like(eL, 2 * d)], -1))
        shifts.append(np.zeros((eL.size, nd)))
        last = e[idx == shape[d] - 1]
        first = last - (shape[d] - 1) * strides[d]
        if periodic[d]:
            ifaces.append(np.stack([last, np.full_like(last, 2 * d + 1), first, np.full_like(last, 2 * d)], -1))
            s = np.zeros((last.size, nd))
            s[:, d] = lengths[d]
            shifts.append(s)
        else:
            bfaces.append(np.stack([first, np.full_like(first, 2 * d), np.full_like(first, 2 * d)], -1))
            bfaces.append(np.stack([last, np.full_like(last, 2 * d + 1), np.full_like(last, 2 * d + 1)], -1))
    return {
        "ndims": nd,
        "etype": "quad" if nd == 2 else "hex",
        "p_g": p_g,
        "nodes": np.ascontiguousarray(nodes, dtype=np.float64),
        "ifaces": np.concatenate(ifaces).astype(np.int32) if ifaces else np.zeros((0, 4), np.int32),
        "shifts": np.concatenate(shifts).astype(np.float64) if shifts else np.zeros((0, nd)),
        "bfaces": np.concatenate(bfaces).astype(np.int32) if bfaces else np.zeros((0, 3), np.int32),
        "lengths": lengths,
        "shape": shape,
    }


def sine_warp(amplitude=0.05):
    """C3's curved-element displacement: the same scalar amplitude*sin x sin y sin z
    added to every coordinate of a node (fixed direction)."""

    def w(X):
        s = amplitude * np.prod(np.sin(X), axis=-1, keepdims=True)
        return np.repeat(s, X.shape[-1], axis=-1)

    return w


def graded_warp(amplitude=0.25):
    """Grading of a periodic box [0, 2 pi]^d with p_g = 1: every coordinate is displaced by amplitude * sin of ITSELF, so the
    elements stay axis-aligned boxes (affine) of different sizes and the periodic images keep matching."""

    def w(X):
        return amplitude * np.sin(X)

    return w


# ----------------------------------------------------------------------------
# unstructured-looking triangle mesh (C4)
# ----------------------------------------------------------------------------
def tri_mesh(n, length=1.0, jitter=0.1, seed=4321, periodic=True):
    """n x n quads on [0,length]^2 split along alternating diagonals; interior
    vertices jittered by U(-jitter*h, jitter*h) per coordinate (seeded); boundary
    vertices unjittered so periodic images match.  Straight-sided (p_g = 1).
    Triangles are counter-clockwise; face k = edge (vertex k -> vertex k+1)."""
    h = length / n
    rng = np.random.default_rng(seed)
    vx, vy = np.meshgrid(np.arange(n + 1) * h, np.arange(n + 1) * h, indexing="xy")  # [j, i]
    V = np.stack([vx, vy], -1)
    jit = rng.uniform(-jitter * h, jitter * h, size=V.shape)
    jit[0, :, :] = 0.0
    jit[-1, :, :] = 0.0
    jit[:, 0, :] = 0.0
    jit[:, -1, :] = 0.0
    V = V + jit

    def vid(i, j):  # vertex id on the (n+1)^2 grid
        return j * (n + 1) + i

    tris = []
    for j in range(n):
        for i in range(n):
            a, b, c, d = vid(i, j), vid(i + 1, j), vid(i + 1, j + 1), vid(i, j + 1)
            if (i + j) % 2 == 0:  # split along (i,j)-(i+1,j+1)
                tris.append((a, b, c))
                tris.append((a, c, d))
            else:  # other diagonal
                tris.append((a, b, d))
                tris.append((b, c, d))
    tris = np.array(tris, dtype=np.int64)
    Vf = V.reshape(-1, 2)
    nodes = Vf[tris]  # [n_el, 3, 2]; p_g=1 lattice order (0,0),(1,0),(0,1) = v0,v1,v2

    # periodic identification of vertex ids
    def canon(v):
        i, j = v % (n + 1), v // (n + 1)
        if periodic:
            i, j = i % n, j % n
        return j * (n + 1) + i

    edges = {}
    for e in range(tris.shape[0]):
        for k in range(3):
            v0, v1 = int(tris[e, k]), int(tris[e, (k + 1) % 3])
            key = tuple(sorted((canon(v0), canon(v1))))
            edges.setdefault(key, []).append((e, k))
    ifaces, shifts, bfaces = [], [], []
    for key, lst in edges.items():
        if len(lst) == 2:
            (eL, fL), (eR, fR) = lst
            mL = 0.5 * (Vf[tris[eL, fL]] + Vf[tris[eL, (fL + 1) % 3]])
            mR = 0.5 * (Vf[tris[eR, fR]] + Vf[tris[eR, (fR + 1) % 3]])
            ifaces.append((eL, fL, eR, fR))
            shifts.append(np.round((mL - mR) / length) * length)
        elif len(lst) == 1:
            (e, f) = lst[0]
            mid = 0.5 * (Vf[tris[e, f]] + Vf[tris[e, (f + 1) % 3]])
            # bc_id: 0 bottom, 1 right, 2 top, 3 left
            tol = 1e-9 * length
            bc = 0 if mid[1] < tol else 1 if mid[0] > length - tol else 2 if mid[1] > length - tol else 3
            bfaces.append((e, f, bc))
        else:
            raise RuntimeError("non-manifold edge")
    return {
        "ndims": 2,
        "etype": "tri",
        "p_g": 1,
        "nodes": np.ascontiguousarray(nodes, dtype=np.float64),
        "ifaces": np.array(ifaces, dtype=np.int32).reshape(-1, 4),
        "shifts": np.array(shifts, dtype=np.float64).reshape(-1, 2),
        "bfaces": np.array(bfaces, dtype=np.int32).reshape(-1, 3),
        "lengths": (length, length),
        "shape": (n, n),
    }


def mixed_mesh(n, length=1.0, jitter=0.1, seed=2468, periodic=True, tri_from=None):
    """Quadrilaterals and triangles sharing edges in one mesh (the paper's mixed unstructured workload): an n x n
    grid on [0,length]^2 whose columns i < tri_from (default n // 2) stay quadrilaterals while the others are split into
    triangles along alternating diagonals; interior vertices jittered by U(-jitter*h, jitter*h) (seeded), boundary vertices
    unjittered so that periodic images match.  Straight-sided (p_g = 1; the jittered quadrilaterals are bilinear, not affine).

    Mixed mesh dictionary:
      ndims 2, parts: [ {etype, p_g, nodes [n_el, n_nodes, 2]} , ... ]   (part 0 = quads, part 1 = triangles)
      ifaces  int32 [n_if, 6] = (partL, elemL, faceL, partR, elemR, faceR)   (order significant, A12)
      shifts  float64 [n_if, 2]:  x_L = x_R + shift
      bfaces  int32 [n_b, 4] = (part, elem, face, bc_id)      bc_id: 0 bottom, 1 right, 2 top, 3 left
    Face numbering per type as in the single-type meshes (quad face = 2 d + s, triangle face k = edge v_k -> v_k+1)."""
    tri_from = n // 2 if tri_from is None else tri_from
    h = length / n
    rng = np.random.default_rng(seed)
    vx, vy = np.meshgrid(np.arange(n + 1) * h, np.arange(n + 1) * h, indexing="xy")
    V = np.stack([vx, vy], -1)
    jit = rng.uniform(-jitter * h, jitter * h, size=V.shape)
    jit[0, :, :] = 0.0
    jit[-1, :, :] = 0.0
    jit[:, 0, :] = 0.0
    jit[:, -1, :] = 0.0
    Vf = (V + jit).reshape(-1, 2)

    def vid(i, j):
        return j * (n + 1) + i

    def canon(v):
        i, j = v % (n + 1), v // (n + 1)
        if periodic:
            i, j = i % n, j % n
        return j * (n + 1) + i

    quads, tris = [], []
    edges = {}

    def add_edge(v0, v1, part, elem, face):
        edges.setdefault(tuple(sorted((canon(v0), canon(v1)))), []).append((part, elem, face, v0, v1))

    for j in range(n):
        for i in range(n):
            a, b, c, d = vid(i, j), vid(i + 1, j), vid(i + 1, j + 1), vid(i, j + 1)
            if i < tri_from:
                e = len(quads)
                quads.append((a, b, d, c))  # lattice order (0,0),(1,0),(0,1),(1,1)
                for face, (v0, v1) in enumerate(((a, d), (b, c), (a, b), (d, c))):  # faces x-, x+, y-, y+
                    add_edge(v0, v1, 0, e, face)
            else:
                pair = ((a, b, c), (a, c, d)) if (i + j) % 2 == 0 else ((a, b, d), (b, c, d))
                for t in pair:
                    e = len(tris)
                    tris.append(t)
                    for k in range(3):
                        add_edge(t[k], t[(k + 1) % 3], 1, e, k)
    ifaces, shifts, bfaces = [], [], []
    tol = 1e-9 * length
    for lst in edges.values():
        if len(lst) == 2:
            (pL, eL, fL, a0, a1), (pR, eR, fR, b0, b1) = lst
            mL, mR = 0.5 * (Vf[a0] + Vf[a1]), 0.5 * (Vf[b0] + Vf[b1])
            ifaces.append((pL, eL, fL, pR, eR, fR))
            shifts.append(np.round((mL - mR) / length) * length)
        elif len(lst) == 1:
            (pt, e, f, a0, a1) = lst[0]
            mid = 0.5 * (Vf[a0] + Vf[a1])
            bc = 0 if mid[1] < tol else 1 if mid[0] > length - tol else 2 if mid[1] > length - tol else 3
            bfaces.append((pt, e, f, bc))
        else:
            raise RuntimeError("non-manifold edge")
    parts = []
    if quads:
        parts.append({"etype": "quad", "p_g": 1, "nodes": np.ascontiguousarray(Vf[np.array(quads)], dtype=np.float64)})
    if tris:
        parts.append({"etype": "tri", "p_g": 1, "nodes": np.ascontiguousarray(Vf[np.array(tris)], dtype=np.float64)})
    if len(parts) == 1:  # degenerate splits keep the part numbering of the interface records consistent
        only = 0 if quads else 1
        ifaces = [(0, eL, fL, 0, eR, fR) for (_, eL, fL, _, eR, fR) in ifaces]
        bfaces = [(0, e, f, bc) for (_, e, f, bc) in bfaces]
        del only
    return {
        "ndims": 2,
        "parts": parts,
        "ifaces": np.array(ifaces, dtype=np.int32).reshape(-1, 6),
        "shifts": np.array(shifts, dtype=np.float64).reshape(-1, 2),
        "bfaces": np.array(bfaces, dtype=np.int32).reshape(-1, 4),
        "lengths": (length, length),
        "shape": (n, n),
    }


def part_mesh(mixed, t):
    """Part t of a mixed mesh as a single-type mesh dictionary: the interfaces whose two sides lie in the part, and the part's
    boundary faces (topology bookkeeping only)."""
    ifc, bf = mixed["ifaces"], mixed["bfaces"]
    own = (ifc[:, 0] == t) & (ifc[:, 3] == t)
    return {
        "ndims": mixed["ndims"], "etype": mixed["parts"][t]["etype"], "p_g": mixed["parts"][t]["p_g"], "nodes": mixed["parts"][t]["nodes"],
        "ifaces": np.ascontiguousarray(ifc[own][:, [1, 2, 4, 5]]), "shifts": np.ascontiguousarray(mixed["shifts"][own]),
        "bfaces": np.ascontiguousarray(bf[bf[:, 0] == t][:, 1:]), "lengths": mixed["lengths"], "shape": mixed["shape"],
    }


def curve_tri_mesh(mesh, p_g=2, amplitude=0.01):
    """Raises a straight-sided triangle mesh to geometry degree p_g: lattice nodes (rows j = 0..p_g, i = 0..p_g-j) of each
    straight triangle, displaced by amplitude*sin(2 pi x/L)*sin(2 pi y/L) in both coordinates (smooth, zero on the box
    boundary, so periodic images and shared edges still match).  Topology unchanged."""
    V = mesh["nodes"]  # [n_el, 3, 2]
    L = np.array(mesh["lengths"])
    pts = []
    for j in range(p_g + 1):
        for i in range(p_g + 1 - j):
            pts.append(V[:, 0] + (i / p_g) * (V[:, 1] - V[:, 0]) + (j / p_g) * (V[:, 2] - V[:, 0]))
    X = np.stack(pts, axis=1)  # [n_el, n_nodes, 2]
    d = amplitude * np.prod(np.sin(2 * np.pi * X / L[None, None, :]), axis=-1, keepdims=True)
    out = dict(mesh)
    out["nodes"] = np.ascontiguousarray(X + np.repeat(d, 2, axis=-1))
    out["p_g"] = p_g
    return out


# ----------------------------------------------------------------------------
# analytic states, evaluated at physical coordinates X[..., nd] -> U[..., nd+2]
# (conserved variables rho, rho*v, E with E = p/(gamma-1) + rho|v|^2/2, Eq 21)
# ----------------------------------------------------------------------------
def _conserved(rho, vel, p, gamma):
    ke = 0.5 * rho * sum(v * v for v in vel)
    return np.stack([rho] + [rho * v for v in vel] + [p / (gamma - 1.0) + ke], axis=-1)


def uniform_state(X, rho=1.0, vel=None, p=1.0, gamma=1.4):
    nd = X.shape[-1]
    vel = (1.0,) * nd if vel is None else vel
    one = np.ones(X.shape[:-1])
    return _conserved(rho * one, [v * one for v in vel], p * one, gamma)


def isentropic_vortex(X, t=0.0, eps=5.0, centre=(5.0, 5.0), vel=(1.0, 1.0), gamma=1.4, period=None):
    """Textbook isentropic vortex, freestream rho=1, (u,v)=vel, p=1.
    `period`: if given, the vortex centre is wrapped so the exact solution on a
    periodic box of that side can be sampled at time t."""
    cx, cy = centre[0] + vel[0] * t, centre[1] + vel[1] * t
    dx, dy = X[..., 0] - cx, X[..., 1] - cy
    if period is not None:
        dx = (dx + 0.5 * period) % period - 0.5 * period
        dy = (dy + 0.5 * period) % period - 0.5 * period
    r2 = dx * dx + dy * dy
    f = eps / (2.0 * np.pi) * np.exp(0.5 * (1.0 - r2))
    u = vel[0] - f * dy
    v = vel[1] + f * dx
    T = 1.0 - (gamma - 1.0) * eps * eps / (8.0 * gamma * np.pi ** 2) * np.exp(1.0 - r2)
    rho = T ** (1.0 / (gamma - 1.0))
    p = rho ** gamma
    return _conserved(rho, [u, v], p, gamma)


def taylor_green(X, mach=0.1, gamma=1.4, rho0=1.0, v0=1.0):
    """Isothermal-variant Taylor-Green vortex; 3-D."""
    x, y, z = X[..., 0], X[..., 1], X[..., 2]
    p0 = rho0 * v0 * v0 / (gamma * mach * mach)
    u = v0 * np.sin(x) * np.cos(y) * np.cos(z)
    v = -v0 * np.cos(x) * np.sin(y) * np.cos(z)
    w = np.zeros_like(x)
    p = p0 + rho0 * v0 * v0 / 16.0 * (np.cos(2 * x) + np.cos(2 * y)) * (np.cos(2 * z) + 2.0)
    rho = rho0 * p / p0
    return _conserved(rho, [u, v, w], p, gamma)


def tgv_viscosity(reynolds=1600.0, rho0=1.0, v0=1.0, length=1.0):
    return rho0 * v0 * length / reynolds


def add_relative_noise(U, rel=1e-3, seed=1234):
    rng = np.random.default_rng(seed)
    return U * (1.0 + rel * rng.uniform(-1.0, 1.0, size=U.shape))


def sinusoidal_2d(X, mach=0.2, gamma=1.4):
    """C4's smooth periodic state on [0,1]^2."""
    x, y = 2 * np.pi * X[..., 0], 2 * np.pi * X[..., 1]
    p0 = 1.0 / (gamma * mach * mach)
    rho = 1.0 + 0.1 * np.sin(x) * np.sin(y)
    u = 1.0 + 0.1 * np.sin(x) * np.cos(y)
    v = 1.0 - 0.1 * np.cos(x) * np.sin(y)
    p = p0 * (1.0 + 0.05 * np.cos(x) * np.cos(y))
    return _conserved(rho, [u, v], p, gamma)


def fourier_state(X, seed, gamma=1.4, mach=0.3, n_modes=8, amp=0.02):
    """C5: freestream rho=1, v=(1,0.5,0.25), p=1/(gamma*mach^2) plus `n_modes`
    low-wavenumber Fourier modes per primitive variable (seeded).  3-D, 2*pi-periodic."""
    rng = np.random.default_rng(seed)
    nd = X.shape[-1]
    free = [1.0, 1.0, 0.5, 0.25][: nd + 1] + [1.0 / (gamma * mach * mach)]
    ks = np.array([(i, j, k) for i in range(-2, 3) for j in range(-2, 3) for k in range(-2, 3) if (i, j, k) != (0, 0, 0)])
    if nd == 2:
        ks = np.array([(i, j) for i in range(-2, 3) for j in range(-2, 3) if (i, j) != (0, 0)])
    prim = []
    for q in range(nd + 2):
        val = np.full(X.shape[:-1], free[q])
        sel = rng.choice(len(ks), size=n_modes, replace=False)
        a = rng.uniform(0.0, amp, size=n_modes) * abs(free[q])
        ph = rng.uniform(0.0, 2 * np.pi, size=n_modes)
        for m in range(n_modes):
            val = val + a[m] * np.cos(X @ ks[sel[m]].astype(float) + ph[m])
        prim.append(val)
    return _conserved(prim[0], prim[1 : 1 + nd], prim[-1], gamma)


# ----------------------------------------------------------------------------
# the BASELINE.json configs
# ----------------------------------------------------------------------------
def config(name, **over):
    """Returns (mesh, disc) for C1..C5 (C5 takes p=, n=, system=) and for Q (768^2 periodic affine quadrilaterals, p=, n=,
    system=: the 2-D tensor-product throughput case of SURVEY 8(f); not a BASELINE.json config).  disc["ref"] is the freestream the state generator of the
    config perturbs (density, velocity, pressure): the library takes it as its constant reference state (a conditioning
    hint, include/fr.h); the oracle ignores it."""
    mesh, disc = _config(name, **over)
    nd = mesh["ndims"]
    p0 = {"C1": 1.0, "C2": 1.0 / (1.4 * 0.1 ** 2), "C3": 1.0 / (1.4 * 0.1 ** 2), "C4": 1.0 / (1.4 * 0.2 ** 2), "C5": 1.0 / (1.4 * 0.3 ** 2), "Q": 1.0 / (1.4 * 0.2 ** 2)}[name]
    v0 = {"C1": (1.0, 1.0), "C2": (0.0,) * 3, "C3": (0.0,) * 3, "C4": (1.0, 1.0), "C5": (1.0, 0.5, 0.25), "Q": (1.0, 1.0)}[name]
    disc["ref"] = dict(rho=1.0, v=v0[:nd], p=p0)
    return mesh, disc


def _config(name, **over):
    g = 1.4
    if name == "C1":
        mesh = box_mesh((8, 8), (10.0, 10.0))
        disc = dict(p=2, system="euler", gamma=g, mu=0.0, Pr=0.71, beta=0.5, tau=0.0, dt=1e-3, steps=10)
    elif name == "C2":
        n = over.get("n", 16)
        mesh = box_mesh((n,) * 3, (2 * np.pi,) * 3)
        disc = dict(p=3, system="navier-stokes", gamma=g, mu=tgv_viscosity(1600.0), Pr=0.71, beta=0.5, tau=0.1, dt=1e-3, steps=20)
    elif name == "C3":
        n = over.get("n", 32)
        p = over.get("p", 4)
        mesh = box_mesh((n,) * 3, (2 * np.pi,) * 3, p_g=p, warp=sine_warp(0.05))
        disc = dict(p=p, system="navier-stokes", gamma=g, mu=tgv_viscosity(1600.0), Pr=0.71, beta=0.5, tau=0.1, dt=1e-3, steps=1)
    elif name == "C4":
        n = over.get("n", 256)
        mesh = tri_mesh(n, 1.0, 0.1, 4321)
        disc = dict(p=3, system="navier-stokes", gamma=g, mu=1.0 / 100.0, Pr=0.71, beta=0.5, tau=0.1, dt=1e-5, steps=1)
    elif name == "C5":
        n = over.get("n", 8)
        p = over.get("p", 3)
        mesh = box_mesh((n,) * 3, (2 * np.pi,) * 3)
        disc = dict(p=p, system=over.get("system", "navier-stokes"), gamma=g, mu=tgv_viscosity(1600.0), Pr=0.71, beta=0.5, tau=0.1, dt=1e-3, steps=1)
    elif name == "Q":
        n = over.get("n", 768)
        mesh = box_mesh((n, n), (1.0, 1.0))
        disc = dict(p=over.get("p", 3), system=over.get("system", "navier-stokes"), gamma=g, mu=1.0 / 100.0, Pr=0.71, beta=0.5, tau=0.1, dt=1e-5, steps=1)
    else:
        raise KeyError(name)
    return mesh, disc


def config_state(name, X, **over):
    """Initial state for a config at solution-point coordinates X[N_u, N_el, nd];
    returns U[N_u, N_V, N_el] (the ABI's [point][var][element] order, unpadded)."""
    if name == "C1":
        U = isentropic_vortex(X)
    elif name == "C2":
        U = taylor_green(X)
    elif name == "C3":
        U = add_relative_noise(taylor_green(X), 1e-3, 1234)
    elif name in ("C4", "Q"):
        U = sinusoidal_2d(X)
    elif name == "C5":
        U = fourier_state(X, seed=2025 + over.get("p", 3))
    else:
        raise KeyError(name)
    return np.ascontiguousarray(np.moveaxis(U, -1, 1))


# ----------------------------------------------------------------------------
# sampling helper for full-size parity: a patch of the mesh around seed elements
# ----------------------------------------------------------------------------
def patch_around(mesh, seeds, hops=2):
    """Sub-mesh made of `seeds` and every element within `hops` face-neighbour steps.

    The RHS of a Navier-Stokes FR element depends on its neighbours' neighbours (compact LDG stencil),
    so on the returned patch the RHS of the SEED elements equals the RHS on the full mesh, whatever the
    boundary condition put on the cut faces (bc_id 0).  Returns (sub_mesh, element ids [n_sub] into the
    full mesh, positions of the seeds inside the patch).  No arithmetic of the method here: topology only.
    """
    ifc = mesh["ifaces"]
    n_el = mesh["nodes"].shape[0]
    inside = np.zeros(n_el, dtype=bool)
    inside[np.asarray(seeds)] = True
    for _ in range(hops):
        touch = inside[ifc[:, 0]] | inside[ifc[:, 2]]
        inside[ifc[touch, 0]] = True
        inside[ifc[touch, 2]] = True
    ids = np.flatnonzero(inside)
    remap = -np.ones(n_el, dtype=np.int64)
    remap[ids] = np.arange(ids.size)
    inL, inR = inside[ifc[:, 0]], inside[ifc[:, 2]]
    both = inL & inR
    sub_if = ifc[both].copy()
    sub_if[:, 0] = remap[sub_if[:, 0]]
    sub_if[:, 2] = remap[sub_if[:, 2]]
    cutL = ifc[inL & ~inR]
    cutR = ifc[inR & ~inL]
    bf = [np.stack([remap[cutL[:, 0]], cutL[:, 1], np.zeros(len(cutL), dtype=np.int64)], -1),
          np.stack([remap[cutR[:, 2]], cutR[:, 3], np.zeros(len(cutR), dtype=np.int64)], -1)]
    old_b = mesh["bfaces"]
    if len(old_b):
        keep = inside[old_b[:, 0]]
        ob = old_b[keep].copy().astype(np.int64)
        ob[:, 0] = remap[ob[:, 0]]
        bf.append(ob)
    sub = dict(mesh)
    sub["nodes"] = np.ascontiguousarray(mesh["nodes"][ids])
    sub["ifaces"] = sub_if.astype(np.int32)
    sub["shifts"] = np.ascontiguousarray(mesh["shifts"][both])
    sub["bfaces"] = np.concatenate(bf).astype(np.int32)
    return sub, ids, remap[np.asarray(seeds)]
