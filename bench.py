#!/usr/bin/env python
"""bench.py — FR RHS throughput (GDOF/s) on B200, one JSON line.

A "step" is one pass of the whole hot path: one fr_rhs evaluation (all seven parts of the north_star)
over the whole synthetic mesh.  Default workload: C3 of BASELINE.json — 32^3 periodic CURVED hexahedra,
p=4, 3-D Navier-Stokes, fp64, Taylor-Green + seeded noise (the configuration the metric's target
"p=4 hexahedral Navier-Stokes FP64 RHS" is quoted on).  Inputs exceed L2 (state 164 MB, working set >1 GB).

  python bench.py [--gpus N] [--steps K] [--warmup W] [--workload C3|C2|C1|C4|C5|Q] [--precision f64|f32]
  python bench.py --impl reference ...      # the oracle on the host cores, bounded sample

Multi-GPU: the path is single-GPU by the north_star ("no sharding or collectives") => replicas only:
every rank runs the same workload; value = N * DOF / max-over-ranks time; scaling "weak".
"""
import argparse
import json
import os
import subprocess
import sys
import threading
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, ROOT)
import workloads as W  # noqa: E402

ORACLE_SINGLE_THREAD_S = None
METRIC = "FR RHS GDOF/s"
UNIT = "GDOF/s"


def parse():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=30)
    ap.add_argument("--warmup", type=int, default=5)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--workload", default="C3")
    ap.add_argument("--precision", default="f64", choices=["f64", "f32"])
    ap.add_argument("--n", type=int, default=0, help="elements per direction (0 = the config's own size)")
    ap.add_argument("--p", type=int, default=0)
    ap.add_argument("--system", default="")
    ap.add_argument("--generic", action="store_true", help="force the generic staged kernels")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--fill", type=float, default=0.0, help="size the mesh so that the device footprint is this fraction of 180 GB (C5)")
    ap.add_argument("--sweep", action="store_true", help="C5 sweep: one JSON line per (p, system, precision) at --fill")
    ap.add_argument("--sweep-p", default="1,2,3,4,5,6")
    ap.add_argument("--sweep-systems", default="navier-stokes,euler")
    ap.add_argument("--sweep-precisions", default="f64,f32")
    ap.add_argument("--peaks", action="store_true", help="measure the FP64 / FP32 FMA peaks and the copy bandwidth of this GPU")
    return ap.parse_args()


def workload(args):
    over = {}
    if args.n:
        over["n"] = args.n
    if args.p:
        over["p"] = args.p
    if args.system:
        over["system"] = args.system
    mesh, disc = W.config(args.workload, **over)
    desc = {
        "workload": "%s: %s %s mesh %s, p=%d, %s, %s, p_g=%d" % (
            args.workload, "x".join(str(s) for s in mesh["shape"]), mesh["etype"],
            "curved periodic" if mesh["p_g"] > 1 else "affine periodic", disc["p"], disc["system"], args.precision, mesh["p_g"]),
        "elements": int(mesh["nodes"].shape[0]),
        "p": disc["p"],
        "system": disc["system"],
        "l2": "inputs larger than L2 (no flush)",
    }
    return mesh, disc, over, desc


# ----------------------------------------------------------------------------------------------
# byte model: SURVEY 8(d) fused lower bound for the whole RHS, and the
# compulsory (read-once / write-once) words per element of each kernel
# ----------------------------------------------------------------------------------------------
def rhs_algorithmic_words(nd, NV, Nu, Nf, ns, affine):
    if ns:
        w = 5 * NV * Nu + 12 * NV * Nf
    else:
        w = 2 * NV * Nu + 4 * NV * Nf  # read U, write R; U^f write + two-sided read, D~ write + read
    if not affine:
        w += (nd * nd + 1) * Nu + (nd + 1) * Nf
    return w


def kernel_bytes(name, nd, NV, Nu, Nf, ns, gfrac=1.0, sz=8, szi=8, affine=False, hex_tma=False):
    """compulsory bytes per element for one launch group (inputs once + outputs once).
    sz: bytes of a state / metric word (8 | 4: the algorithmic size in the context's precision); szi: bytes of a flux-point /
    gradient intermediate as the path stores it (= sz on the hexahedral TMA path, 8 elsewhere); index words are 4 bytes,
    gather offsets 8.  gfrac: fraction of the faces that carry an LDG weight (1/2 when |beta| = 1/2)."""
    # NOTE: fp_n (own normals, read by the gradient kernels) is counted at nd * N_f words whatever the mesh
    met = (nd * nd + 1) * Nu * sz
    if affine and (name.startswith("hex_") or name.startswith("el_")):
        met = (nd * nd + 1) * sz  # straight-sided elements: the fused kernels read the metric terms of ONE point per element
    pair_tab = (4 * 4 + (nd + 2) * sz) * Nf // 2  # per flux-point pair: 4 indices, unit normal, two J n
    if affine and hex_tma:  # affine hexahedra on the TMA path: normal and J n per FACE (fr_dev.hpp: pf_n), indices per pair
        pair_tab = 4 * 4 * Nf // 2 + 2 * nd * (nd + 1) * sz
    U, R = Nu * NV * sz, Nu * NV * sz
    t = {
        # generic staged path (App A sequence)
        "apply_M0": U + Nf * NV * szi,
        "common_sol": 2 * Nf * NV * szi + 4 * 4 * Nf // 2,
        "apply_M46_M6": U + (Nf + nd * Nu) * NV * szi,
        "grad_phys": 2 * nd * Nu * NV * szi + met,
        "apply_M5": nd * (Nu + Nf) * NV * szi,
        "tflux": U + (2 if ns else 1) * nd * Nu * NV * szi + nd * nd * Nu * sz,
        "common_flux": (2 + (nd if ns else 0)) * Nf * NV * szi + pair_tab,
        "apply_M132_M3_negdivconf": (nd * Nu + Nf) * NV * szi + R + Nu * sz,
        # quadrilateral line kernels (fr_tensor.cu)
        "tp_interp": U + Nf * NV * szi,
        "tp_interp_q": nd * (Nu + Nf) * NV * szi,
        "tp_grad": U + Nf * NV * szi + met + nd * Nu * NV * szi,
        "tp_div": (nd * Nu + Nf) * NV * szi + R + Nu * sz,
        # TMA-pipelined hexahedral path (fr_hex_interp_tma.cu, fr_hex_tma.cu, fr_hex_fluxdiv_tma.cu)
        "hex_interp_tma": U + Nf * NV * szi,
        # U, partner U^f and its offset (faces with an LDG weight), S, 1/J, own normals -> G^f, Q
        "hex_gradface": U + 2 * gfrac * Nf * NV * szi + gfrac * Nf * 8 + met + gfrac * nd * Nf * sz + nd * Nu * NV * szi,
        "common_flux_g": (2 + gfrac) * Nf * NV * szi + pair_tab,      # U^f, G^f -> D~ (in place), normals, J n
        "hex_fluxdiv_tma": U + R + Nf * NV * szi + (nd * Nu * NV * szi if ns else 0) + met,
        # fused triangle / quadrilateral kernels (fr_element.cu)
        "el_interp": U + Nf * NV * szi,
        # U, own and partner U^f (+ 8-byte offsets, side codes), S, 1/J, normals -> Q, G^f
        "el_gradface": U + 3 * Nf * NV * szi + Nf * 9 + met + nd * Nf * sz + nd * Nu * NV * szi,
        "el_fluxdiv": U + R + Nf * NV * szi + (nd * Nu * NV * szi if ns else 0) + met,
    }
    return t.get(name)


def max_over_ranks(ms, world, device="cuda"):
    """Timed-region duration = max over ranks (the only cross-rank exchange of the replicas-only N>1 path)."""
    if world <= 1:
        return float(ms)
    import torch
    import torch.distributed as dist

    t = torch.tensor([ms], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def aggregate_value(dof, ms_step, world):
    """Whole-job GDOF/s: every rank processed `dof` per step (weak scaling, replicas)."""
    return world * dof / (ms_step * 1e-3) / 1e9


class ClockSampler(threading.Thread):
    def __init__(self, index):
        super().__init__(daemon=True)
        self.index, self.stop_flag, self.rows = index, False, []

    def run(self):
        q = "clocks.sm,clocks.max.sm,clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap"
        while not self.stop_flag:
            try:
                out = subprocess.run(["nvidia-smi", "-i", str(self.index), "--query-gpu=" + q, "--format=csv,noheader,nounits"],
                                     capture_output=True, text=True, timeout=5).stdout.strip()
                if out:
                    self.rows.append([x.strip() for x in out.split(",")])
            except Exception:
                pass
            time.sleep(0.1)

    def summary(self):
        sm = [float(r[0]) for r in self.rows if r[0].replace(".", "").isdigit()]
        mx = [float(r[1]) for r in self.rows if r[1].replace(".", "").isdigit()]
        reasons = set()
        for r in self.rows:
            for name, v in zip(["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"], r[2:6]):
                if v.lower().startswith("active"):
                    reasons.add(name)
        return {"sm_mhz": float(np.median(sm)) if sm else None, "sm_max_mhz": max(mx) if mx else None, "reasons": sorted(reasons), "samples": len(sm)}


def time_oracle(args, sample_n, reps):
    """The oracle as it stands on the host cores, on a bounded sample of the workload's shape."""
    from oracle.fr_oracle import FROracle

    a2 = argparse.Namespace(**vars(args))
    if sample_n:
        a2.n = sample_n
    mesh, disc, over, _ = workload(a2)
    o = FROracle(mesh, disc)
    U = W.config_state(args.workload, np.asarray(o.xu_phys, float), **over)
    o.rhs(U)
    ts = []
    for _ in range(reps):
        t0 = time.perf_counter()
        o.rhs(U)
        ts.append(time.perf_counter() - t0)
    global ORACLE_SINGLE_THREAD_S
    try:
        from threadpoolctl import threadpool_info, threadpool_limits

        cores = max([i.get("num_threads", 1) for i in threadpool_info()] + [1])
        with threadpool_limits(limits=1):  # the same code with its BLAS calls on one thread
            t0 = time.perf_counter()
            o.rhs(U)
            ORACLE_SINGLE_THREAD_S = time.perf_counter() - t0
    except Exception:
        cores = os.cpu_count()
        ORACLE_SINGLE_THREAD_S = None
    return U.size, ts, cores, "%s %s (%d elements, %d DOF), %d oracle RHS evaluations, numpy float64" % (
        args.workload, ("at full size, %s" if not sample_n else "on its %s version") % "x".join(str(s) for s in mesh["shape"]), mesh["nodes"].shape[0], U.size, reps)


def sample_size(args):
    """Elements per direction of the oracle's timed sample: C1, C2 and C4 at full size, C3 on its 16^3
    version (1/8 of the elements, same shape), C5 on the 8^3 sub-problem; scaled per DOF."""
    return {"C3": 16, "C5": 8, "Q": 64}.get(args.workload, 0)


def run_reference(args):
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    dof, ts, cores, sample = time_oracle(args, sample_size(args), max(args.steps, 1) + args.warmup)
    ts = ts[args.warmup:]
    ms = 1e3 * float(np.mean(ts))
    val = dof / (ms * 1e-3) / 1e9
    _, _, _, desc = workload(args)
    desc["sample"] = sample
    out = {
        "impl": "reference", "metric": METRIC, "value": val, "unit": UNIT, "n_gpus": args.gpus, "steps": len(ts), "warmup": args.warmup,
        "ms_per_step": ms, "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": desc,
        "cpu_baseline": {"value": val, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": sample, "cpu": cpu_model(),
                         "single_thread_value": (dof / ORACLE_SINGLE_THREAD_S / 1e9) if ORACLE_SINGLE_THREAD_S else None},
        "e2e": {"value": val, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }
    print(json.dumps(out))


def fill_size(args, fraction, hbm_bytes=180e9):
    """Elements per direction of the periodic cube whose device footprint (u, rhs, RHS scratch, RK4 registers, the library's own
    tables) is `fraction` of the HBM, from the library's own size queries on a small probe mesh; capped so that the host-side
    setup (mesh arrays, coordinates, lookup tables: measured ~ (600 + 170 N_f + 60 N_u) bytes per element at peak) stays inside
    the box's free memory."""
    from paper_1312_1638_b200 import Context
    from paper_1312_1638_b200.binding import FLAG_HOST_ONLY

    a2 = argparse.Namespace(**vars(args))
    a2.n = 4
    mesh, disc, _, _ = workload(a2)
    ctx = Context(mesh).setup_operators(precision=args.precision, **disc)
    ld = ctx.ld
    sz = 8 if args.precision == "f64" else 4
    # pair indices, per-face normals / J n (affine hexahedra), own normals + partner offsets, face codes, metric terms of one point
    tables = ctx.Nf / 2 * 16 + 24 * sz + ctx.Nf * (3 * sz + 8) + 6 + 10 * sz
    per_elem = (2 * ctx.state_bytes + ctx.workspace_bytes) / ld + tables
    ctx.teardown()
    n_dev = int((fraction * hbm_bytes / per_elem) ** (1.0 / 3.0))
    host_per_elem = 600 + 170 * ctx.Nf + 60 * ctx.Nu + 2 * ctx.Nu * ctx.NV * sz
    try:
        avail = [int(l.split()[1]) * 1024 for l in open("/proc/meminfo") if l.startswith("MemAvailable")][0]
    except Exception:
        avail = 64e9
    n_host = int((0.55 * avail / host_per_elem) ** (1.0 / 3.0))
    return min(n_dev, n_host), per_elem, n_dev, n_host


def measure(args, world, rank, local, barrier, light=False):
    """One workload: device-resident timing, end to end with host buffers, per-kernel events, RK4 step; returns the JSON dict
    (rank 0) or None.  light: no end-to-end leg and no CPU baseline (sweeps at 90 GB)."""
    import torch

    from paper_1312_1638_b200 import Context
    from paper_1312_1638_b200.binding import FLAG_FORCE_GENERIC, FLAG_LEAN

    mesh, disc, over, desc = workload(args)
    t0 = time.time()
    flags = (FLAG_FORCE_GENERIC if args.generic else 0) | (FLAG_LEAN if light else 0)
    ctx = Context(mesh).setup_operators(precision=args.precision, flags=flags, **disc)
    setup_s = time.time() - t0
    n_el_mesh, p_g = int(mesh["nodes"].shape[0]), mesh["p_g"]
    if light:
        mesh = None  # release the host mesh
    X = ctx.solution_point_coords()
    U = ctx.pad(W.config_state(args.workload, X, **over))
    del X
    dof = ctx.Nu * ctx.NV * ctx.n_elems
    u_host = torch.from_numpy(U)
    if not light:
        u_host = u_host.pin_memory()
        r_host = torch.empty_like(u_host).pin_memory()
    u = u_host.cuda()
    if light:
        del u_host, U
    r = torch.zeros_like(u)
    work = torch.zeros(ctx.workspace_bytes, dtype=torch.uint8, device="cuda")
    stream = torch.cuda.current_stream().cuda_stream
    up, rp, wp = u.data_ptr(), r.data_ptr(), work.data_ptr()
    dev_bytes = int(torch.cuda.memory_allocated())

    # ---- device-resident timing ----
    for _ in range(max(args.warmup, 3)):
        ctx.rhs(up, rp, wp, stream)
    barrier()
    sampler = ClockSampler(local)
    sampler.start()
    ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    ev0.record()
    for _ in range(args.steps):
        ctx.rhs(up, rp, wp, stream)
    ev1.record()
    barrier()
    ms_total = ev0.elapsed_time(ev1)
    # keep the GPU busy a little longer if the timed region was too short for a clock sample
    t_end = time.time() + max(0.0, 0.6 - ms_total * 1e-3)
    while time.time() < t_end:
        ctx.rhs(up, rp, wp, stream)
        torch.cuda.synchronize()
    sampler.stop_flag = True
    sampler.join()
    ms_step = max_over_ranks(ms_total, world) / args.steps
    value = aggregate_value(dof, ms_step, world)

    # ---- end to end through the C ABI with host buffers (H2D + RHS + D2H per step) ----
    e2e = None
    if not light:
        n_e2e = max(3, min(args.steps, 10))
        for _ in range(2):
            ctx.rhs_host(u_host.data_ptr(), r_host.data_ptr(), up, rp, wp, stream)
        barrier()
        ev0.record()
        for _ in range(n_e2e):
            ctx.rhs_host(u_host.data_ptr(), r_host.data_ptr(), up, rp, wp, stream)
        ev1.record()
        barrier()
        e2e_ms = max_over_ranks(ev0.elapsed_time(ev1), world) / n_e2e
        e2e = {"value": aggregate_value(dof, e2e_ms, world), "unit": UNIT, "ms_per_step": e2e_ms,
               "h2d_bytes_per_step": int(u_host.numel() * u_host.element_size()), "d2h_bytes_per_step": int(r_host.numel() * r_host.element_size())}

    # ---- per-kernel durations (events between kernels, same stream), dominant kernel roofline ----
    acc = {}
    n_prof = max(3, min(args.steps, 10))
    for _ in range(n_prof):
        for name, ms in ctx.rhs_profiled(up, rp, wp, stream):
            acc[name] = acc.get(name, 0.0) + ms / n_prof
    if rank != 0:
        return None
    peaks = {}
    pk_path = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(pk_path):
        peaks = json.load(open(pk_path))
    peak_gbs = float(peaks.get("hbm_gbs", 6650.0))
    peak_src = "measured (MEASURED_PEAKS.json hbm_gbs)" if "hbm_gbs" in peaks else "fallback 6650 GB/s"
    nd, NV, Nu, Nf, ns = ctx.ndims, ctx.NV, ctx.Nu, ctx.Nf, disc["system"] == "navier-stokes"
    affine = p_g == 1
    sz = 8 if args.precision == "f64" else 4
    szi = sz if any(n.startswith("hex_") for n in acc) else 8  # the hexahedral TMA path stores its intermediates in the storage precision
    kern = []
    for name, ms in acc.items():
        byt = kernel_bytes(name, nd, NV, Nu, Nf, ns, 0.5 if abs(abs(disc.get("beta", 0.5)) - 0.5) < 1e-15 else 1.0, sz, szi, affine,
                           hex_tma=any(n.startswith("hex_") for n in acc))
        gbs = (byt * ctx.n_elems / (ms * 1e-3) / 1e9) if (byt and ms > 0) else None
        kern.append({"name": name, "ms": ms, "share": ms / sum(acc.values()), "algorithmic_GBps": gbs})
    kern.sort(key=lambda k: -k["ms"])
    top = kern[0]
    traffic = None
    tpath = os.path.join(ROOT, "profiles", "traffic.json")
    lib = os.path.join(ROOT, "paper_1312_1638_b200", "libfr_b200.so")
    if os.path.exists(tpath):
        try:
            t = json.load(open(tpath))
            # the ncu figures belong to one build of the library: dropped when the sources have changed since
            if t.get("source_sha16") == source_sha16():
                traffic = t.get(args.workload + "-" + args.precision, {}).get(top["name"])
        except Exception:
            traffic = None
    roofline = {"bound": "hbm", "kernel": top["name"], "achieved": top["algorithmic_GBps"], "peak": peak_gbs, "unit": "GB/s",
                "frac": (top["algorithmic_GBps"] / peak_gbs) if top["algorithmic_GBps"] else None, "traffic": traffic,
                "peak_source": peak_src, "kernel_ms": top["ms"], "kernel_share_of_step": top["share"]}
    words = rhs_algorithmic_words(nd, NV, Nu, Nf, ns, affine)
    rhs_gbs = words * sz * ctx.n_elems / (ms_step * 1e-3) / 1e9
    out = {
        "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": max(args.warmup, 3),
        "ms_per_step": ms_step, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
        "dtype": args.precision, "data": "synthetic",
        "config": dict(desc, parallelism="replicas only (%d)" % world, setup_s=round(setup_s, 2), device_bytes=dev_bytes),
        "clocks": sampler.summary(),
        "e2e": e2e,
        "gpu_launches": int(ctx.rhs_kernel_launches) * args.steps,
        "roofline": roofline,
        "rhs_roofline": {"bound": "hbm", "algorithmic_bytes_per_point": words * sz / Nu,
                         "achieved": rhs_gbs, "peak": peak_gbs, "unit": "GB/s", "frac": rhs_gbs / peak_gbs,
                         "note": "SURVEY 8(d) fused lower-bound bytes of the WHOLE RHS / measured RHS time"},
        "kernels": kern,
        "s_per_rk4_step": None,
    }
    # RK4 step time
    for _ in range(2):
        ctx.rk4_step(up, 1e-6, wp, stream)
    torch.cuda.synchronize()
    ev0.record()
    nrk = 5
    for _ in range(nrk):
        ctx.rk4_step(up, 1e-6, wp, stream)
    ev1.record()
    torch.cuda.synchronize()
    out["s_per_rk4_step"] = ev0.elapsed_time(ev1) * 1e-3 / nrk
    if not light and not args.no_cpu_baseline and world == 1:
        cdof, ts, cores, sample = time_oracle(args, sample_size(args), 5)
        out["cpu_baseline"] = {"value": cdof / float(np.mean(ts)) / 1e9, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": sample,
                               "cpu": cpu_model(), "single_thread_value": (cdof / ORACLE_SINGLE_THREAD_S / 1e9) if ORACLE_SINGLE_THREAD_S else None}
    else:
        out["cpu_baseline"] = None
    ctx.teardown()
    del u, r, work
    torch.cuda.empty_cache()
    return out


def source_sha16():
    """hash of the CUDA sources: profiles/traffic.json records the one its ncu figures were taken with"""
    import hashlib

    h = hashlib.sha256()
    d = os.path.join(ROOT, "paper_1312_1638_b200", "csrc")
    for f in sorted(os.listdir(d)):
        h.update(open(os.path.join(d, f), "rb").read())
    return h.hexdigest()[:16]


def cpu_model():
    try:
        return [l.split(":", 1)[1].strip() for l in open("/proc/cpuinfo") if l.startswith("model name")][0]
    except Exception:
        return "unknown"


def run_peaks(args):
    """Measured roofline denominators of this GPU: FP64 / FP32 FMA peaks (the library's microbenchmark) and copy bandwidth."""
    import torch

    from paper_1312_1638_b200.binding import measure_peaks

    torch.cuda.set_device(int(os.environ.get("LOCAL_RANK", "0")))
    out = measure_peaks()
    out["gpu"] = torch.cuda.get_device_name()
    pk = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(pk):
        out["driver_hbm_gbs"] = json.load(open(pk)).get("hbm_gbs")
    print(json.dumps(out))


def main():
    args = parse()
    if args.impl == "reference":
        return run_reference(args)
    if args.peaks:
        return run_peaks(args)

    import torch
    import torch.distributed as dist

    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device: the FR library has no CPU fallback")
    torch.cuda.set_device(local)
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    if args.sweep:
        # C5 of BASELINE.json: p = 1..6 x {Navier-Stokes, Euler} x {f64, f32} on meshes sized to --fill of the HBM
        args.workload = "C5"
        ps = [int(x) for x in args.sweep_p.split(",")]
        for p in ps:
            for system in args.sweep_systems.split(","):
                for prec in args.sweep_precisions.split(","):
                    a2 = argparse.Namespace(**vars(args))
                    a2.p, a2.system, a2.precision = p, system, prec
                    a2.n, per_elem, n_dev, n_host = fill_size(a2, args.fill)
                    out = measure(a2, world, rank, local, barrier, light=True)
                    if out is not None:
                        out["config"].update(fill_target=args.fill, device_bytes_per_element=per_elem, n_for_fill=n_dev, n_host_cap=n_host)
                        print(json.dumps(out), flush=True)
    else:
        if args.fill > 0:
            args.n = fill_size(args, args.fill)[0]
        out = measure(args, world, rank, local, barrier, light=args.fill > 0)
        if out is not None:
            print(json.dumps(out))
    if world > 1:
        dist.destroy_process_group()


if __name__ == "__main__":
    main()
