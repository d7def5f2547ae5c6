"""Pins for the mixed-element oracle (FRMixedOracle): what fixes the expected values is the
single-type oracle (already pinned) on meshes where both apply, the analytic Navier-Stokes divergence (sympy), and the
invariants of the scheme -- never the mixed oracle's own formulas."""
import numpy as np
import pytest

import workloads as W
from oracle.fr_oracle import FRMixedOracle, FROracle, flux_inviscid
from test_oracle_rhs import _analytic_ns_rhs

NS = dict(system="navier-stokes", gamma=1.4, mu=0.02, Pr=0.71, beta=0.5, tau=0.1)


def _coords(o):
    return [np.asarray(q.xu_phys, float) for q in o.parts]


def _states(o, fn, noise=0.0, seed=3):
    out = []
    for i, X in enumerate(_coords(o)):
        U = fn(X)
        if noise:
            U = W.add_relative_noise(U, noise, seed + i)
        out.append(np.ascontiguousarray(np.moveaxis(U, -1, 1)))
    return out


def split_single_type(mesh, mask):
    """A single-type mesh cut into two parts of the SAME type (elements with mask True -> part 1): topology bookkeeping only."""
    part = mask.astype(np.int64)
    local = np.where(mask, np.cumsum(mask) - 1, np.cumsum(~mask) - 1)
    ifc, bf = mesh["ifaces"], mesh["bfaces"]
    parts = [{"etype": mesh["etype"], "p_g": mesh["p_g"], "nodes": np.ascontiguousarray(mesh["nodes"][part == t])} for t in (0, 1)]
    i6 = np.stack([part[ifc[:, 0]], local[ifc[:, 0]], ifc[:, 1], part[ifc[:, 2]], local[ifc[:, 2]], ifc[:, 3]], -1)
    b4 = np.stack([part[bf[:, 0]], local[bf[:, 0]], bf[:, 1], bf[:, 2]], -1) if len(bf) else np.zeros((0, 4))
    return {"ndims": mesh["ndims"], "parts": parts, "ifaces": i6.astype(np.int32), "shifts": mesh["shifts"], "bfaces": b4.astype(np.int32),
            "lengths": mesh["lengths"], "shape": mesh["shape"]}, part, local


@pytest.mark.parametrize("kind", ["quad", "tri"])
@pytest.mark.parametrize("system", ["euler", "navier-stokes"])
def test_two_parts_of_one_type_equal_the_single_type_oracle(kind, system):
    """Cutting a single-type mesh into two parts changes only the lookup table: the mixed oracle must
    reproduce the single-type oracle's right-hand side element by element, with boundary faces present."""
    mesh = W.box_mesh((5, 4), (1.0, 1.0), p_g=2, warp=W.sine_warp(0.03), periodic=(True, False)) if kind == "quad" else W.tri_mesh(4, 1.0, 0.1, 5, periodic=False)
    bcs = {0: ("sup-inflow", dict(rho=1.0, v=(1.0, 0.5), p=17.8)), 1: ("sub-outflow", dict(p=17.0)),
           2: ("noslip-wall", dict(cpTw=60.0, v=(0.2, 0.0))), 3: ("noslip-wall", dict(cpTw=62.0, v=(0.0, 0.0)))}
    prm = dict(NS, p=3, system=system)
    o1 = FROracle(mesh, prm, bcs)
    n_el = mesh["nodes"].shape[0]
    mask = np.random.default_rng(1).random(n_el) < 0.5
    mixed, part, local = split_single_type(mesh, mask)
    o2 = FRMixedOracle(mixed, prm, bcs)
    X = np.asarray(o1.xu_phys, float)
    U = np.ascontiguousarray(np.moveaxis(W.add_relative_noise(W.sinusoidal_2d(X), 1e-2, 9), -1, 1))
    R1 = o1.rhs(U)
    R2 = o2.rhs([np.ascontiguousarray(U[:, :, part == t]) for t in (0, 1)])
    for t in (0, 1):
        assert np.max(np.abs(R2[t] - R1[:, :, part == t])) <= 1e-13 * np.max(np.abs(R1))


@pytest.mark.parametrize("system", ["euler", "navier-stokes"])
@pytest.mark.parametrize("p", [1, 3])
def test_mixed_freestream_and_conservation(system, p):
    mesh = W.mixed_mesh(6, 1.0, 0.1)
    o = FRMixedOracle(mesh, dict(NS, p=p, system=system))
    U0 = _states(o, lambda X: W.uniform_state(X, rho=1.0, vel=(1.0, 0.5), p=1.0))
    fmax = max(np.max(np.abs(flux_inviscid(np.moveaxis(u, 1, 0), 1.4))) for u in U0)
    h = 1.0 / 6
    assert max(np.max(np.abs(r)) for r in o.rhs(U0)) <= 1e-12 * fmax * 2 / h
    R = o.rhs(_states(o, W.sinusoidal_2d, noise=1e-2))
    tot, mag = o.integrate(R), o.integrate([np.abs(r) for r in R])
    assert np.all(np.abs(tot) <= 1e-12 * mag) and np.all(mag > 1e-3)


def test_mixed_rhs_converges_to_analytic_navier_stokes():
    """Spectral convergence of the mixed discretisation to the symbolic Navier-Stokes divergence (sympy), in both parts."""
    mu, Pr = 0.05, 0.71
    fU, fR = _analytic_ns_rhs(2, mu, Pr)
    errs = []
    for p in (3, 6, 9):
        mesh = W.mixed_mesh(6, 2 * np.pi, 0.1, 7)
        o = FRMixedOracle(mesh, dict(p=p, system="navier-stokes", gamma=1.4, mu=mu, Pr=Pr, beta=0.5, tau=0.1))
        Us, Ex = [], []
        for X in _coords(o):
            args = [X[..., d] for d in range(2)]
            Us.append(np.stack([np.broadcast_to(a, X.shape[:-1]) for a in fU(*args)], 1))
            Ex.append(np.stack([np.broadcast_to(a, X.shape[:-1]) for a in fR(*args)], 1))
        R = o.rhs(Us)
        scale = np.max([np.max(np.abs(e), axis=(0, 2)) for e in Ex], axis=0)[None, :, None]
        errs.append(max(np.max(np.abs(r - e) / scale) for r, e in zip(R, Ex)))
    assert errs[0] > errs[1] > errs[2] and errs[0] / errs[2] > 50 and errs[2] < 2e-3, errs


def test_interface_records_must_cover_every_flux_point():
    mesh = W.mixed_mesh(4)
    bad = dict(mesh, ifaces=mesh["ifaces"][1:], shifts=mesh["shifts"][1:])
    with pytest.raises(ValueError):
        FRMixedOracle(bad, dict(NS, p=2))
