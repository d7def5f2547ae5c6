"""CPU-side checks of the C-ABI library: it loads, exports every symbol include/fr.h declares, its
host operator builder and mesh setup agree with the oracle (no CUDA call is made: FR_FLAG_HOST_ONLY),
and its error paths return codes instead of crashing."""
import ctypes as C
import os
import re

import numpy as np
import pytest

import workloads as W
from oracle.fr_oracle import FROracle

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def fr():
    import paper_1312_1638_b200.binding as b

    return b


def test_exports_every_declared_symbol(fr):
    hdr = open(os.path.join(ROOT, "include", "fr.h")).read()
    declared = set(re.findall(r"\b(fr_[a-z0-9_]+)\s*\(", hdr))
    assert len(declared) >= 20
    raw = C.CDLL(fr.LIB_PATH)
    for name in declared:
        assert hasattr(raw, name), name
    assert declared == set(fr.EXPORTS)


def test_build_targets_sm_100a():
    src = open(os.path.join(ROOT, "paper_1312_1638_b200", "build.py")).read()
    assert "arch=compute_100a,code=sm_100a" in src


CASES = [("C1", {}), ("C2", dict(n=3)), ("C3", dict(n=3, p=4)), ("C3", dict(n=2, p=2)), ("C4", dict(n=6)), ("C5", dict(n=2, p=6)),
         ("C1", dict(correction="sd")), ("C1", dict(correction="hu")), ("C2", dict(n=2, correction="hu")), ("C5", dict(n=2, p=5, correction="sd"))]


@pytest.mark.parametrize("name,over", CASES)
def test_host_tables_match_oracle(fr, name, over):
    """M0..M6 (DG, SD and HU correction functions: the library builds the family of the paper's ref [10] from its parameter c,
    the oracle from the closed forms), metrics, coordinates and the pair set."""
    over = dict(over)
    corr = over.pop("correction", "dg")
    mesh, disc = W.config(name, **over)
    disc = dict(disc, correction=corr)
    ctx = fr.Context(mesh).setup_operators(flags=fr.FLAG_HOST_ONLY, **disc)
    o = FROracle(mesh, disc)
    ops = o.ops
    for i, M in enumerate([ops.M0, ops.M1, ops.M2, ops.M3, ops.M4, ops.M5, ops.M6]):
        A, B = ctx.get_operator(i), np.asarray(M, dtype=np.float64)
        assert A.shape == B.shape
        assert np.max(np.abs(A - B)) <= 4e-16 * max(1.0, np.max(np.abs(B))), "M%d" % i
    assert np.max(np.abs(ctx.solution_point_coords() - np.asarray(o.xu_phys, float))) < 1e-14 * max(mesh["lengths"])
    s, r = ctx.get_metrics()
    So = np.moveaxis(np.asarray(o.Su, float), (2, 3), (0, 1)).reshape(o.nd * o.nd, o.Nu, o.Nel)
    assert np.max(np.abs(s[:, :, : o.Nel] - So)) <= 1e-15 * np.max(np.abs(So))
    assert np.max(np.abs(r[:, : o.Nel] * np.asarray(o.Ju, float) - 1)) <= 1e-15
    pairs, nrm, jn = ctx.get_pairs()
    mine = set(map(tuple, pairs.tolist()))
    theirs = set(zip(o.pL_s.tolist(), o.pL_e.tolist(), o.pR_s.tolist(), o.pR_e.tolist()))
    assert mine == theirs
    assert np.allclose(nrm, np.asarray(o.nhat_f, float)[pairs[:, 0], pairs[:, 1]], atol=1e-15)
    assert np.allclose(jn[:, 0], np.asarray(o.Jn_f, float)[pairs[:, 0], pairs[:, 1]], rtol=1e-15)
    assert np.allclose(jn[:, 1], np.asarray(o.Jn_f, float)[pairs[:, 2], pairs[:, 3]], rtol=1e-15)
    # iteration order: sorted by the L flux point
    key = pairs[:, 0].astype(np.int64) * o.Nel + pairs[:, 1]
    assert np.all(np.diff(key) > 0)
    assert ctx.ld % 16 == 0 and ctx.ld >= o.Nel


def test_error_codes(fr):
    mesh, disc = W.config("C1")
    # NULL context
    assert fr.lib.fr_num_solution_points(None) < 0
    assert fr.lib.fr_rhs(None, None, None, None, None) == -1
    fr.lib.fr_teardown(None)
    # queries before fr_setup_operators
    ctx = fr.Context(mesh)
    assert fr.lib.fr_num_flux_points(ctx._h) < 0
    assert b"fr_setup_operators" in fr.lib.fr_last_error(ctx._h)
    # bad discretisation
    with pytest.raises(fr.FrError):
        ctx.setup_operators(p=2, system="euler", gamma=0.9, flags=fr.FLAG_HOST_ONLY)
    # host-only context refuses to run
    ctx.setup_operators(flags=fr.FLAG_HOST_ONLY, **disc)
    assert fr.lib.fr_rhs(ctx._h, 1, 2, 3, None) == -1
    # inverted element (J < 0)
    bad = dict(mesh, nodes=mesh["nodes"][:, ::-1, :].copy())
    with pytest.raises(fr.FrError) as ei:
        fr.Context(bad).setup_operators(flags=fr.FLAG_HOST_ONLY, **disc)
    assert ei.value.code == -2
    # a face listed twice / a face never listed
    dup = dict(mesh, ifaces=np.concatenate([mesh["ifaces"], mesh["ifaces"][:1]]), shifts=np.concatenate([mesh["shifts"], mesh["shifts"][:1]]))
    with pytest.raises(fr.FrError):
        fr.Context(dup).setup_operators(flags=fr.FLAG_HOST_ONLY, **disc)
    miss = dict(mesh, ifaces=mesh["ifaces"][1:], shifts=mesh["shifts"][1:])
    with pytest.raises(fr.FrError):
        fr.Context(miss).setup_operators(flags=fr.FLAG_HOST_ONLY, **disc)
    # wrong periodic shift -> unmatched flux points
    wrong = dict(mesh, shifts=mesh["shifts"] * 0.5)
    with pytest.raises(fr.FrError) as ei:
        fr.Context(wrong).setup_operators(flags=fr.FLAG_HOST_ONLY, **disc)
    assert ei.value.code == -2
    # mismatched ndims / etype
    with pytest.raises(fr.FrError):
        fr.Context(dict(mesh, ndims=3))
