"""Thin ctypes binding of libfr_b200.so (include/fr.h).  Argument marshalling only: every step of the
FR right-hand side runs in the library's CUDA kernels.  There is no CPU fallback: if the shared
library is missing, importing this module raises.

PyTorch appears only in the callers (tests, bench.py) to allocate device memory and streams; this
module takes raw device pointers (ints) so it works with any allocator.
"""
import ctypes as C
import os

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libfr_b200.so")

QUAD, TRI, HEX = 0, 1, 2
EULER, NAVIER_STOKES = 0, 1
F32, F64 = 0, 1
BC_SUP_INFLOW, BC_SUB_OUTFLOW, BC_NOSLIP_WALL = 0, 1, 2
FLAG_FORCE_GENERIC, FLAG_HOST_ONLY, FLAG_LEAN = 1, 2, 4
STATIC_WORK_BYTES = 32 * 1024 * 1024  # FR_STATIC_WORK_BYTES: scratch of fr_rhs_static, held inside the library
CORRECTIONS = {"dg": 0, "sd": 1, "hu": 2}
STEPPERS = {"euler": 0, "rk4": 1, "dopri5": 2}
ETYPES = {"quad": QUAD, "tri": TRI, "hex": HEX}
SYSTEMS = {"euler": EULER, "navier-stokes": NAVIER_STOKES}
BC_KINDS = {"sup-inflow": BC_SUP_INFLOW, "sub-outflow": BC_SUB_OUTFLOW, "noslip-wall": BC_NOSLIP_WALL}


class FrError(RuntimeError):
    def __init__(self, code, text):
        super().__init__("fr error %d: %s" % (code, text))
        self.code = code


class fr_bc_desc(C.Structure):
    _fields_ = [("kind", C.c_int32), ("rho", C.c_double), ("v", C.c_double * 3), ("p", C.c_double), ("cpTw", C.c_double)]


class fr_mesh_desc(C.Structure):
    _fields_ = [
        ("ndims", C.c_int32), ("etype", C.c_int32), ("p_g", C.c_int32), ("n_bcs", C.c_int32),
        ("n_elems", C.c_int64), ("n_ifaces", C.c_int64), ("n_bfaces", C.c_int64),
        ("nodes", C.c_void_p), ("ifaces", C.c_void_p), ("shifts", C.c_void_p), ("bfaces", C.c_void_p), ("bcs", C.c_void_p),
    ]


class fr_mesh_part(C.Structure):
    _fields_ = [("etype", C.c_int32), ("p_g", C.c_int32), ("n_elems", C.c_int64), ("nodes", C.c_void_p)]


class fr_mixed_mesh_desc(C.Structure):
    _fields_ = [
        ("ndims", C.c_int32), ("n_parts", C.c_int32), ("n_bcs", C.c_int32), ("reserved", C.c_int32),
        ("n_ifaces", C.c_int64), ("n_bfaces", C.c_int64),
        ("parts", C.c_void_p), ("ifaces", C.c_void_p), ("shifts", C.c_void_p), ("bfaces", C.c_void_p), ("bcs", C.c_void_p),
    ]


class fr_part_info_t(C.Structure):
    _fields_ = [("etype", C.c_int32), ("reserved", C.c_int32), ("n_elems", C.c_int64), ("n_solution_points", C.c_int64),
                ("n_flux_points", C.c_int64), ("leading_dim", C.c_int64), ("state_offset", C.c_int64)]


class fr_disc_desc(C.Structure):
    _fields_ = [
        ("p", C.c_int32), ("system", C.c_int32), ("precision", C.c_int32), ("flags", C.c_int32),
        ("correction", C.c_int32), ("reserved", C.c_int32),
        ("gamma", C.c_double), ("mu", C.c_double), ("Pr", C.c_double), ("ldg_beta", C.c_double), ("ldg_tau", C.c_double),
        ("rho_ref", C.c_double), ("v_ref", C.c_double * 3), ("p_ref", C.c_double),
    ]


def _load():
    if not os.path.exists(LIB_PATH):
        raise ImportError(
            "libfr_b200.so is missing (%s): build it with `python -m paper_1312_1638_b200.build`; there is no CPU fallback" % LIB_PATH
        )
    lib = C.CDLL(LIB_PATH)
    P, I64 = C.c_void_p, C.c_int64
    sig = {
        "fr_setup_mesh": (C.c_int, [C.POINTER(P), C.POINTER(fr_mesh_desc)]),
        "fr_setup_mesh_mixed": (C.c_int, [C.POINTER(P), C.POINTER(fr_mixed_mesh_desc)]),
        "fr_num_parts": (I64, [P]),
        "fr_part_info": (C.c_int, [P, C.c_int, C.POINTER(fr_part_info_t)]),
        "fr_part_solution_point_coords": (C.c_int, [P, C.c_int, P]),
        "fr_setup_operators": (C.c_int, [P, C.POINTER(fr_disc_desc)]),
        "fr_num_solution_points": (I64, [P]), "fr_num_flux_points": (I64, [P]), "fr_num_vars": (I64, [P]),
        "fr_num_pairs": (I64, [P]), "fr_leading_dim": (I64, [P]), "fr_state_bytes": (I64, [P]),
        "fr_workspace_bytes": (I64, [P]), "fr_rhs_kernel_launches": (I64, [P]),
        "fr_stepper_workspace_bytes": (I64, [P, C.c_int]),
        "fr_euler_step": (C.c_int, [P, P, C.c_double, P, P]),
        "fr_dopri5_step": (C.c_int, [P, P, C.c_double, P, P, P]),
        "fr_solution_point_coords": (C.c_int, [P, P]),
        "fr_operator_dims": (C.c_int, [P, C.c_int, C.POINTER(I64), C.POINTER(I64)]),
        "fr_get_operator": (C.c_int, [P, C.c_int, P]),
        "fr_get_pairs": (C.c_int, [P, P, P, P]),
        "fr_get_metrics": (C.c_int, [P, P, P]),
        "fr_rhs": (C.c_int, [P, P, P, P, P]),
        "fr_rhs_static": (C.c_int, [P, P, P, P]),
        "fr_rhs_profiled": (C.c_int, [P, P, P, P, P, C.c_int, C.POINTER(C.c_int), P, P]),
        "fr_rk4_step": (C.c_int, [P, P, C.c_double, P, P]),
        "fr_rhs_host": (C.c_int, [P, P, P, P, P, P, P]),
        "fr_state_lincomb": (C.c_int, [P, C.c_int, C.POINTER(C.c_void_p), C.POINTER(C.c_double), P, P]),
        "fr_measure_peaks": (C.c_int, [C.POINTER(C.c_double), C.POINTER(C.c_double), C.POINTER(C.c_double)]),
        "fr_teardown": (None, [P]),
        "fr_last_error": (C.c_char_p, [P]),
    }
    for name, (res, args) in sig.items():
        fn = getattr(lib, name)
        fn.restype, fn.argtypes = res, args
    return lib


lib = _load()
EXPORTS = ["fr_setup_mesh", "fr_setup_mesh_mixed", "fr_num_parts", "fr_part_info", "fr_part_solution_point_coords", "fr_setup_operators", "fr_num_solution_points", "fr_num_flux_points", "fr_num_vars", "fr_num_pairs",
           "fr_leading_dim", "fr_state_bytes", "fr_workspace_bytes", "fr_stepper_workspace_bytes", "fr_rhs_kernel_launches",
           "fr_euler_step", "fr_dopri5_step", "fr_solution_point_coords",
           "fr_operator_dims", "fr_get_operator", "fr_get_pairs", "fr_get_metrics", "fr_rhs", "fr_rhs_static", "fr_rhs_profiled", "fr_rk4_step", "fr_rhs_host", "fr_state_lincomb",
           "fr_measure_peaks", "fr_teardown", "fr_last_error"]


def measure_peaks():
    """-> dict(fp64_tflops, fp32_tflops, copy_gbs) of the current CUDA device (fr_measure_peaks)."""
    a, b, c = C.c_double(), C.c_double(), C.c_double()
    rc = lib.fr_measure_peaks(C.byref(a), C.byref(b), C.byref(c))
    if rc != 0:
        raise FrError(rc, "fr_measure_peaks failed")
    return {"fp64_tflops": a.value, "fp32_tflops": b.value, "copy_gbs": c.value}


def _ptr(a):
    return a.ctypes.data_as(C.c_void_p) if a is not None and a.size else None


class Context:
    """Owns one fr_ctx.  Method names mirror the C entry points."""

    def __init__(self, mesh, bcs=None):
        """mesh: workloads.py mesh dict; bcs: {bc_id: (kind, params)} as the oracle takes them."""
        self._h = C.c_void_p()
        self._keep = []
        self.mixed = "parts" in mesh
        if self.mixed:
            return self._init_mixed(mesh, bcs)
        nodes = np.ascontiguousarray(mesh["nodes"], dtype=np.float64)
        ifaces = np.ascontiguousarray(mesh["ifaces"], dtype=np.int32)
        shifts = np.ascontiguousarray(mesh["shifts"], dtype=np.float64)
        bfaces = np.ascontiguousarray(mesh["bfaces"], dtype=np.int32)
        bcs = bcs or {}
        nb = (max(bcs) + 1) if bcs else 0
        arr = (fr_bc_desc * max(nb, 1))()
        for i, (kind, par) in bcs.items():
            arr[i].kind = BC_KINDS[kind]
            arr[i].rho = float(par.get("rho", 0.0))
            v = list(par.get("v", ())) + [0.0] * 3
            for d in range(3):
                arr[i].v[d] = float(v[d])
            arr[i].p = float(par.get("p", 0.0))
            arr[i].cpTw = float(par.get("cpTw", 0.0))
        for i in range(nb):
            if i not in bcs:
                arr[i].kind = BC_SUP_INFLOW
        d = fr_mesh_desc(
            ndims=mesh["ndims"], etype=ETYPES[mesh["etype"]], p_g=mesh["p_g"], n_bcs=nb,
            n_elems=nodes.shape[0], n_ifaces=ifaces.shape[0], n_bfaces=bfaces.shape[0],
            nodes=_ptr(nodes), ifaces=_ptr(ifaces), shifts=_ptr(shifts), bfaces=_ptr(bfaces),
            bcs=C.cast(arr, C.c_void_p) if nb else None,
        )
        rc = lib.fr_setup_mesh(C.byref(self._h), C.byref(d))
        if rc != 0:
            raise FrError(rc, (lib.fr_last_error(None) or b"").decode())
        self.ndims, self.n_elems = mesh["ndims"], nodes.shape[0]

    @staticmethod
    def _bc_array(bcs):
        bcs = bcs or {}
        nb = (max(bcs) + 1) if bcs else 0
        arr = (fr_bc_desc * max(nb, 1))()
        for i, (kind, par) in bcs.items():
            arr[i].kind = BC_KINDS[kind]
            arr[i].rho = float(par.get("rho", 0.0))
            v = list(par.get("v", ())) + [0.0] * 3
            for d in range(3):
                arr[i].v[d] = float(v[d])
            arr[i].p = float(par.get("p", 0.0))
            arr[i].cpTw = float(par.get("cpTw", 0.0))
        return arr, nb

    def _init_mixed(self, mesh, bcs):
        """mesh: workloads.mixed_mesh dictionary (parts of one element type each, 6-column interface records)."""
        nodes = [np.ascontiguousarray(p["nodes"], dtype=np.float64) for p in mesh["parts"]]
        parts = (fr_mesh_part * len(nodes))()
        for t, (p, nd_) in enumerate(zip(mesh["parts"], nodes)):
            parts[t].etype, parts[t].p_g, parts[t].n_elems, parts[t].nodes = ETYPES[p["etype"]], p["p_g"], nd_.shape[0], _ptr(nd_)
        ifaces = np.ascontiguousarray(mesh["ifaces"], dtype=np.int32)
        shifts = np.ascontiguousarray(mesh["shifts"], dtype=np.float64)
        bfaces = np.ascontiguousarray(mesh["bfaces"], dtype=np.int32)
        arr, nb = self._bc_array(bcs)
        d = fr_mixed_mesh_desc(ndims=mesh["ndims"], n_parts=len(nodes), n_bcs=nb, n_ifaces=ifaces.shape[0], n_bfaces=bfaces.shape[0],
                               parts=C.cast(parts, C.c_void_p), ifaces=_ptr(ifaces), shifts=_ptr(shifts), bfaces=_ptr(bfaces),
                               bcs=C.cast(arr, C.c_void_p) if nb else None)
        rc = lib.fr_setup_mesh_mixed(C.byref(self._h), C.byref(d))
        if rc != 0:
            raise FrError(rc, (lib.fr_last_error(None) or b"").decode())
        self.ndims, self.n_elems = mesh["ndims"], sum(n.shape[0] for n in nodes)

    def _check(self, rc):
        if rc != 0:
            raise FrError(rc, (lib.fr_last_error(self._h) or b"").decode())

    def setup_operators(self, p, system, precision="f64", gamma=1.4, mu=0.0, Pr=0.71, beta=0.5, tau=0.1, flags=0, correction="dg",
                        ref=None, **_):
        """ref: optional constant reference state dict(rho=, v=(..), p=) (fr.h: conditioning hint)."""
        d = fr_disc_desc(p=p, system=SYSTEMS[system], precision=F64 if precision in ("f64", F64) else F32, flags=flags,
                         correction=CORRECTIONS[correction], gamma=gamma, mu=mu, Pr=Pr, ldg_beta=beta, ldg_tau=tau)
        if ref:
            d.rho_ref, d.p_ref = float(ref["rho"]), float(ref["p"])
            for i, v in enumerate(ref.get("v", ())):
                d.v_ref[i] = float(v)
        self._check(lib.fr_setup_operators(self._h, C.byref(d)))
        self.dtype = np.float64 if d.precision == F64 else np.float32
        self.NV = lib.fr_num_vars(self._h)
        if self.mixed:
            self.parts = []
            for t in range(lib.fr_num_parts(self._h)):
                info = fr_part_info_t()
                self._check(lib.fr_part_info(self._h, t, C.byref(info)))
                self.parts.append(dict(etype=info.etype, n_elems=info.n_elems, Nu=info.n_solution_points, Nf=info.n_flux_points,
                                       ld=info.leading_dim, offset=info.state_offset))
            return self
        self.Nu = lib.fr_num_solution_points(self._h)
        self.Nf = lib.fr_num_flux_points(self._h)
        self.NV = lib.fr_num_vars(self._h)
        self.ld = lib.fr_leading_dim(self._h)
        self.dtype = np.float64 if d.precision == F64 else np.float32
        return self

    num_pairs = property(lambda self: lib.fr_num_pairs(self._h))
    state_bytes = property(lambda self: lib.fr_state_bytes(self._h))
    workspace_bytes = property(lambda self: lib.fr_workspace_bytes(self._h))
    rhs_kernel_launches = property(lambda self: lib.fr_rhs_kernel_launches(self._h))

    def solution_point_coords(self):
        if self.mixed:
            out = []
            for t, p in enumerate(self.parts):
                x = np.empty((p["Nu"], p["n_elems"], self.ndims), dtype=np.float64)
                self._check(lib.fr_part_solution_point_coords(self._h, t, _ptr(x)))
                out.append(x)
            return out
        x = np.empty((self.Nu, self.n_elems, self.ndims), dtype=np.float64)
        self._check(lib.fr_solution_point_coords(self._h, _ptr(x)))
        return x

    def get_operator(self, i):
        r, c = C.c_int64(), C.c_int64()
        self._check(lib.fr_operator_dims(self._h, i, C.byref(r), C.byref(c)))
        m = np.empty((r.value, c.value), dtype=np.float64)
        self._check(lib.fr_get_operator(self._h, i, _ptr(m)))
        return m

    def get_pairs(self):
        n = self.num_pairs
        pairs = np.empty((n, 4), dtype=np.int32)
        nrm = np.empty((n, self.ndims), dtype=np.float64)
        jn = np.empty((n, 2), dtype=np.float64)
        self._check(lib.fr_get_pairs(self._h, _ptr(pairs), _ptr(nrm), _ptr(jn)))
        return pairs, nrm, jn

    def get_metrics(self):
        s = np.empty((self.ndims * self.ndims, self.Nu, self.ld), dtype=np.float64)
        r = np.empty((self.Nu, self.ld), dtype=np.float64)
        self._check(lib.fr_get_metrics(self._h, _ptr(s), _ptr(r)))
        return s, r

    # --- the hot path: raw device pointers (ints) in, nothing out ---
    def rhs(self, u_ptr, rhs_ptr, work_ptr, stream=0):
        self._check(lib.fr_rhs(self._h, u_ptr, rhs_ptr, work_ptr, stream))

    def rhs_static(self, u_ptr, rhs_ptr, stream=0):
        """fr_rhs with the scratch in the library's static device array (no allocation; at most STATIC_WORK_BYTES; calls that
        overlap on the GPU race, include/fr.h)."""
        self._check(lib.fr_rhs_static(self._h, u_ptr, rhs_ptr, stream))

    def rhs_profiled(self, u_ptr, rhs_ptr, work_ptr, stream=0):
        """-> [(kernel name, ms)] for one RHS (events between kernels; synchronises)."""
        n = C.c_int()
        ms = (C.c_float * 32)()
        names = C.create_string_buffer(32 * 32)
        self._check(lib.fr_rhs_profiled(self._h, u_ptr, rhs_ptr, work_ptr, stream, 32, C.byref(n), C.cast(ms, C.c_void_p), C.cast(names, C.c_void_p)))
        return [(names.raw[32 * i : 32 * i + 32].split(b"\0")[0].decode(), float(ms[i])) for i in range(n.value)]

    def rk4_step(self, u_ptr, dt, work_ptr, stream=0):
        self._check(lib.fr_rk4_step(self._h, u_ptr, float(dt), work_ptr, stream))

    def stepper_workspace_bytes(self, stepper):
        return lib.fr_stepper_workspace_bytes(self._h, STEPPERS[stepper])

    def euler_step(self, u_ptr, dt, work_ptr, stream=0):
        self._check(lib.fr_euler_step(self._h, u_ptr, float(dt), work_ptr, stream))

    def dopri5_step(self, u_ptr, dt, work_ptr, stream=0, err_ptr=None):
        self._check(lib.fr_dopri5_step(self._h, u_ptr, float(dt), work_ptr, stream, err_ptr))

    def state_lincomb(self, in_ptrs, coefs, out_ptr, stream=0):
        """out = sum coefs[i] * in[i] over state matrices (device pointers)."""
        n = len(in_ptrs)
        arr = (C.c_void_p * n)(*in_ptrs)
        cf = (C.c_double * n)(*[float(x) for x in coefs])
        self._check(lib.fr_state_lincomb(self._h, n, arr, cf, out_ptr, stream))

    def rhs_host(self, u_host_ptr, rhs_host_ptr, u_ptr, rhs_ptr, work_ptr, stream=0):
        self._check(lib.fr_rhs_host(self._h, u_host_ptr, rhs_host_ptr, u_ptr, rhs_ptr, work_ptr, stream))

    # --- layout helpers (host side, no arithmetic of the method) ---
    def pad(self, u):
        """[Nu, NV, n_elems] -> padded [Nu, NV, ld] in the context precision (pad columns zero).
        Mixed meshes: list of such arrays, one per part -> ONE flat buffer with the parts at their state offsets."""
        if self.mixed:
            flat = np.zeros(self.state_bytes // np.dtype(self.dtype).itemsize, dtype=self.dtype)
            for p, up in zip(self.parts, u):
                o = p["offset"] // flat.itemsize
                flat[o:o + p["Nu"] * self.NV * p["ld"]].reshape(p["Nu"], self.NV, p["ld"])[:, :, : p["n_elems"]] = up
            return flat
        out = np.zeros((self.Nu, self.NV, self.ld), dtype=self.dtype)
        out[:, :, : self.n_elems] = u
        return out

    def unpad(self, u):
        u = np.asarray(u)
        if self.mixed:
            out = []
            for p in self.parts:
                o = p["offset"] // u.itemsize
                out.append(np.array(u.reshape(-1)[o:o + p["Nu"] * self.NV * p["ld"]].reshape(p["Nu"], self.NV, p["ld"])[:, :, : p["n_elems"]]))
            return out
        return u.reshape(self.Nu, self.NV, self.ld)[:, :, : self.n_elems]

    def teardown(self):
        if self._h:
            lib.fr_teardown(self._h)
            self._h = C.c_void_p()

    def __del__(self):
        try:
            self.teardown()
        except Exception:
            pass
