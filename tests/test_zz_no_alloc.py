"""fr_rhs_static (include/fr.h): the right-hand side with its scratch in the library's static device array, for callers that
cannot allocate device memory.  Checked against the existing path (fr_rhs with a caller-owned workspace) on the same inputs,
on calls in a row that share the array across states, contexts, element types and precisions.  Collected last on purpose
(file name): the suite runs with pytest -x.  Needs no other test to have run before it."""
import numpy as np
import pytest

import workloads as W
from _util import rel_l2_per_field, rel_max_per_field

pytestmark = pytest.mark.gpu

TOL64, TOL32 = 1e-12, 1e-5  # the bars of test_gpu_parity.py
NS = dict(system="navier-stokes", gamma=1.4, mu=0.02, Pr=0.71, beta=0.5, tau=0.1)


class _Case:
    """One context with its buffers: u, the result of fr_rhs (caller-owned workspace) and the result of fr_rhs_static."""

    def __init__(self, mesh, disc, precision="f64", bcs=None):
        import torch

        from paper_1312_1638_b200 import Context

        self.torch = torch
        self.ctx = ctx = Context(mesh, bcs).setup_operators(precision=precision, **disc)
        self.tol = TOL64 if precision == "f64" else TOL32
        td = torch.float64 if precision == "f64" else torch.float32
        n = ctx.state_bytes // np.dtype(ctx.dtype).itemsize
        self.u = torch.zeros(n, dtype=td, device="cuda")
        self.r_ref = torch.zeros(n, dtype=td, device="cuda")
        self.r_new = torch.zeros(n, dtype=td, device="cuda")
        self.work = torch.zeros(max(ctx.workspace_bytes, 256), dtype=torch.uint8, device="cuda")
        self.stream = torch.cuda.current_stream().cuda_stream

    def state(self, seed):
        """sinusoidal (2-D) / Taylor-Green (3-D) state with seeded relative noise, at the context's solution points"""
        ctx = self.ctx
        X = ctx.solution_point_coords()
        gen = W.sinusoidal_2d if ctx.ndims == 2 else W.taylor_green
        if ctx.mixed:
            U = [np.ascontiguousarray(np.moveaxis(W.add_relative_noise(gen(x), 1e-2, seed + i), -1, 1)) for i, x in enumerate(X)]
        else:
            U = np.ascontiguousarray(np.moveaxis(W.add_relative_noise(gen(X), 1e-2, seed), -1, 1))
        self.u.copy_(self.torch.from_numpy(np.ascontiguousarray(ctx.pad(U)).reshape(-1)))

    def compare(self, label, seed):
        torch, ctx = self.torch, self.ctx
        self.state(seed)
        self.r_ref.fill_(float("nan"))
        self.r_new.fill_(float("nan"))
        ctx.rhs(self.u.data_ptr(), self.r_ref.data_ptr(), self.work.data_ptr(), self.stream)
        torch.cuda.synchronize()
        free0 = torch.cuda.mem_get_info()[0]
        ctx.rhs_static(self.u.data_ptr(), self.r_new.data_ptr(), self.stream)
        torch.cuda.synchronize()
        free1 = torch.cuda.mem_get_info()[0]
        ref, got = ctx.unpad(self.r_ref.cpu().numpy()), ctx.unpad(self.r_new.cpu().numpy())
        if not ctx.mixed:
            ref, got = [ref], [got]
        for t, (a, b) in enumerate(zip(got, ref)):
            assert np.all(np.isfinite(a)) and np.all(np.isfinite(b)), label
            assert np.max(np.abs(b)) > 1e-3, label  # a right-hand side that is not trivially zero
            err, emax = rel_l2_per_field(a, b), rel_max_per_field(a, b)
            print("%s part %d: fr_rhs_static vs fr_rhs rel-L2 per field %s, max-abs %s" % (label, t, err, emax))
            assert np.all(err <= self.tol), (label, err)
            assert np.all(emax <= 30 * self.tol), (label, emax)
        return free0, free1


def _hex(precision):
    mesh, disc = W.config("C3", n=3, p=3)  # curved hexahedra, Navier-Stokes: the TMA kernels of the C3 path
    return _Case(mesh, disc, precision)


def test_static_scratch_matches_fr_rhs_on_calls_in_a_row():
    from paper_1312_1638_b200.binding import STATIC_WORK_BYTES

    a = _hex("f64")
    assert a.ctx.stepper_workspace_bytes("euler") < STATIC_WORK_BYTES
    a.compare("hex-f64 call 1", 11)
    free0, free1 = a.compare("hex-f64 call 2", 12)  # second call in a row: another state, the array holds the first call's scratch
    assert free0 == free1, "fr_rhs_static changed the free device memory: %d -> %d" % (free0, free1)
    # other contexts, layouts and precisions over the same array, then the first context again
    b = _hex("f32")
    b.compare("hex-f32", 13)
    tri = _Case(W.tri_mesh(6, 1.0, 0.1, 5), dict(NS, p=3, ref=dict(rho=1.0, v=(1.0, 1.0), p=1.0 / (1.4 * 0.2 ** 2))))
    tri.compare("tri-f64", 14)
    mixed = _Case(W.mixed_mesh(5, 1.0, 0.1), dict(NS, p=2, ref=dict(rho=1.0, v=(1.0, 1.0), p=1.0 / (1.4 * 0.2 ** 2))))
    mixed.compare("mixed-f64", 15)
    euler = _Case(*W.config("C1"))  # Euler on quadrilaterals
    euler.compare("quad-euler-f64", 16)
    a.compare("hex-f64 call 3", 17)
    for c in (a, b, tri, mixed, euler):
        c.ctx.teardown()


def test_static_scratch_rejects_contexts_beyond_its_size():
    from paper_1312_1638_b200 import Context, FrError
    from paper_1312_1638_b200.binding import STATIC_WORK_BYTES

    import torch

    mesh, disc = W.config("C5", n=16, p=4)
    ctx = Context(mesh).setup_operators(**disc)
    reg = -(-ctx.state_bytes // 256) * 256
    need = ctx.stepper_workspace_bytes("euler") - reg  # scratch of the right-hand side alone
    assert need > STATIC_WORK_BYTES, need
    u = torch.ones(ctx.state_bytes // 8, dtype=torch.float64, device="cuda")
    r = torch.full_like(u, 7.0)
    with pytest.raises(FrError) as ei:
        ctx.rhs_static(u.data_ptr(), r.data_ptr(), torch.cuda.current_stream().cuda_stream)
    msg = str(ei.value)
    assert "FR_STATIC_WORK_BYTES" in msg and str(need) in msg and str(STATIC_WORK_BYTES) in msg, msg
    torch.cuda.synchronize()
    assert bool(torch.all(r == 7.0))  # nothing was launched
    ctx.teardown()
