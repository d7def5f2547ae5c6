"""Shared helpers for the parity tests (host-side marshalling only)."""
import numpy as np


def rel_l2_per_field(a, b):
    """||a-b||_2 / ||b||_2 per variable; arrays [Nu, NV, Nel]."""
    a = np.asarray(a, dtype=np.longdouble)
    b = np.asarray(b, dtype=np.longdouble)
    num = np.sqrt(np.sum((a - b) ** 2, axis=(0, 2)))
    den = np.sqrt(np.sum(b ** 2, axis=(0, 2)))
    return np.asarray(num / den, dtype=np.float64)


def rel_max_per_field(a, b):
    """max|a-b| / max|b| per variable (the max-abs companion of the L2 norm)."""
    a = np.asarray(a, dtype=np.longdouble)
    b = np.asarray(b, dtype=np.longdouble)
    return np.asarray(np.max(np.abs(a - b), axis=(0, 2)) / np.max(np.abs(b), axis=(0, 2)), dtype=np.float64)


# parity triples of the current pytest session (written to gpurun_out/parity_records.jsonl by conftest.py)
RECORDS = []


class GpuRunner:
    """Allocates device buffers with torch and calls the C-ABI through the binding."""

    def __init__(self, ctx):
        import torch

        self.torch = torch
        self.ctx = ctx
        self.tdtype = torch.float64 if ctx.dtype == np.float64 else torch.float32
        n = ctx.state_bytes // np.dtype(ctx.dtype).itemsize  # flat buffers: one matrix, or the parts of a mixed mesh
        self.u = torch.zeros(n, dtype=self.tdtype, device="cuda")
        self.r = torch.zeros(n, dtype=self.tdtype, device="cuda")
        self.work = torch.zeros(max(ctx.stepper_workspace_bytes("dopri5"), 256), dtype=torch.uint8, device="cuda")
        self.stream = torch.cuda.current_stream().cuda_stream

    def set_state(self, U):
        self.u.copy_(self.torch.from_numpy(np.ascontiguousarray(self.ctx.pad(U)).reshape(-1)))

    def rhs(self, U=None):
        if U is not None:
            self.set_state(U)
        self.r.fill_(float("nan"))
        self.ctx.rhs(self.u.data_ptr(), self.r.data_ptr(), self.work.data_ptr(), self.stream)
        self.torch.cuda.synchronize()
        return self.ctx.unpad(self.r.cpu().numpy())

    def rk4(self, U, dt, steps, stepper="rk4"):
        self.set_state(U)
        step = {"rk4": self.ctx.rk4_step, "euler": self.ctx.euler_step, "dopri5": self.ctx.dopri5_step}[stepper]
        for _ in range(steps):
            step(self.u.data_ptr(), dt, self.work.data_ptr(), self.stream)
        self.torch.cuda.synchronize()
        return self.ctx.unpad(self.u.cpu().numpy())

    def dopri5(self, U, dt):
        """one DOPRI5 step -> (new state, RMS of the embedded error estimate)"""
        self.set_state(U)
        err = self.torch.zeros(1, dtype=self.torch.float64, device="cuda")
        self.ctx.dopri5_step(self.u.data_ptr(), dt, self.work.data_ptr(), self.stream, err.data_ptr())
        self.torch.cuda.synchronize()
        return self.ctx.unpad(self.u.cpu().numpy()), float(err.item())
