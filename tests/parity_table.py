"""Writes the per-field parity table: for every BASELINE.json config the relative
L2 distance, per conserved variable, of
    (a) the GPU result (through the C ABI)      from the oracle run in long double,
    (b) the oracle run in plain double           from the oracle run in long double   (the rounding floor of the problem),
next to the bar of the tests.  Calls only oracle/ and the C-ABI binding.  Needs a CUDA device.

    python tests/parity_table.py profiles/r02_parity.md
"""
import os
import sys
import time

import numpy as np

HERE = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, os.path.dirname(HERE))
sys.path.insert(0, HERE)

import workloads as W  # noqa: E402
import test_gpu_parity as T  # noqa: E402
from _util import GpuRunner, rel_l2_per_field, rel_max_per_field  # noqa: E402
from oracle.fr_oracle import FROracle  # noqa: E402

FIELDS2, FIELDS3 = ["rho", "rho u", "rho v", "E"], ["rho", "rho u", "rho v", "rho w", "E"]


def fmt(v):
    return " ".join("%.1e" % x for x in np.atleast_1d(v))


def row(out, label, got, o, U, sel=None, f32=False):
    """one table row; f32: inputs already rounded, bar 1e-5, floor not needed"""
    t0 = time.time()
    R = o.rhs(np.asarray(U, dtype=np.float64))
    R_ld = T._ld(o, np.asarray(U, dtype=np.float64), sel)
    Rs = R if sel is None else R[:, :, sel]
    e_gpu, e_dbl, e_max = rel_l2_per_field(got, R_ld), rel_l2_per_field(Rs, R_ld), rel_max_per_field(got, R_ld)
    tol = T.TOL32 if f32 else T.TOL64
    bar = np.maximum(tol, 2 * e_dbl)
    ok = bool(np.all(e_gpu <= bar))
    meets = bool(np.all(e_gpu <= tol))
    out.append("| %s | %s | %s | %s | %s | %s | %s |" % (label, fmt(e_gpu), fmt(e_dbl), fmt(e_max), "%.0e" % tol,
                                                        "yes" if meets else "NO (%s)" % ("within 2x floor" if ok else "ABOVE BAR"), "%.0fs" % (time.time() - t0)))
    print(out[-1], flush=True)


def main(path):
    import torch

    out = ["# Parity table, round 2: GPU vs the oracle in long double, per conserved variable",
           "",
           "Written by `python tests/parity_table.py %s` on %s (%s)." % (path, time.strftime("%Y-%m-%d"), torch.cuda.get_device_name(0)),
           "Columns: relative L2 error per field (order %s; 2-D cases have no `rho w`) of the GPU result against the" % ", ".join(FIELDS3),
           "long-double oracle; the same for the oracle in plain double (the rounding floor of the problem, SURVEY A16);",
           "max-abs error of the GPU result relative to the field's max; the north_star tolerance; whether every field meets it.",
           "",
           "| case | GPU vs long double | double oracle vs long double | GPU max-abs / max | tol | all fields <= tol | oracle time |",
           "|---|---|---|---|---|---|---|"]
    # C1, C2, C4 in full
    for name in ("C1", "C2", "C4"):
        mesh, disc = W.config(name)
        o = FROracle(mesh, disc)
        U = W.config_state(name, np.asarray(o.xu_phys, float))
        row(out, "%s full (%d elements, p=%d, %s, fp64)" % (name, mesh["nodes"].shape[0], disc["p"], disc["system"]),
            GpuRunner(T._ctx(mesh, disc)).rhs(U), o, U)
    # C3 at full size, sampled elements
    for prec in ("f64", "f32"):
        got, seeds, o, Usub, pos = T.sampled_full_size("C3", prec)
        row(out, "C3 32^3 curved p=4 NS, %d sampled elements, %s" % (seeds.size, prec), got[:, :, seeds], o, Usub, sel=pos, f32=prec == "f32")
    # C5 shapes at 8^3
    for p in range(1, 7):
        for system in ("navier-stokes", "euler"):
            n = 8 if p <= 4 else 6
            mesh, disc = W.config("C5", n=n, p=p, system=system)
            o = FROracle(mesh, disc)
            U = W.config_state("C5", np.asarray(o.xu_phys, float), p=p)
            for prec in ("f64", "f32"):
                Uin = U if prec == "f64" else U.astype(np.float32)
                got = GpuRunner(T._ctx(mesh, disc, precision=prec)).rhs(Uin)
                row(out, "C5 %d^3 affine p=%d %s %s" % (n, p, system, prec), got, o, Uin, f32=prec == "f32")
    with open(path, "w") as f:
        f.write("\n".join(out) + "\n")


if __name__ == "__main__":
    main(sys.argv[1] if len(sys.argv) > 1 else "gpurun_out/parity_table.md")
