#!/usr/bin/env python
"""bench.py -- throughput of the domain-wall hot path on B200.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl reference]

One "step" = one pass of the whole hot path over one batch of seeded synthetic input on the
16^3 x 32 x Ls=16 fp32 workload (BASELINE.json configs[2]/[3]):
    a1 import+export (1 field) | a2-a4 D_hop, D_DW, H_DW, D_PV at nrhs=1 and D_DW at nrhs=12, 48 |
    a5/a6 Schur M_pc on 4 RHS | a7 axpy/inner/norm2 (12 RHS) | a8 order-64 Chebyshev on 24 vectors |
    a9 20 red-black CG iterations.
metric = GFlop/s in the standard convention of 1320 flop per 5D site per D_hop-bearing operator
apply (R20), summed over every apply in the step.  Rank 0 prints ONE JSON line; `detail` carries the
per-row numbers (D_DW GB/s and GFlop/s per nrhs, Chebyshev vectors/s, CG iterations/s).
N > 1: independent replicas (the path does not shard: DESIGN.md sec. 8), one process per GPU.
"""
from __future__ import annotations

import argparse
import json
import os
import statistics
import subprocess
import sys
import threading
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

L = (16, 16, 16, 32)
LS, M5, MASS = 16, 1.8, 0.01
V5 = L[0] * L[1] * L[2] * L[3] * LS
FLOP_PER_SITE = 1320.0
CHEB_ORDER, CHEB_NVEC, CHEB_LO, CHEB_HI = 64, 24, 0.01, 70.0
CG_ITERS = 20
# dram__bytes_read.sum + dram__bytes_write.sum per launch of the dominant kernel (ncu --set full; average of the two
# epilogue variants): parsed from the ncu summary below (lines "traffic_bytes_per_launch: ..." and "commit: ..."), so that
# the number always names the capture and the commit it was taken at
NCU_TRAFFIC_SOURCE = "profiles/r2_cheb_traffic.md"
WORKLOAD = "16^3x32xLs16 fp32: D_hop/D_DW/H_DW/D_PV (nrhs 1,12,48) + Schur(4) + BLAS-1 + order-64 Chebyshev(24) + 20 rb-CG it"


def peaks():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        return json.load(open(p)).get("hbm_gbs", 6650.0), "measured (MEASURED_PEAKS.json hbm_gbs)"
    return 6650.0, "fallback (B200_PROFILING.md 6.65 TB/s)"


def ncu_traffic():
    """(bytes per launch or None, source string) from NCU_TRAFFIC_SOURCE."""
    import re
    path = os.path.join(ROOT, NCU_TRAFFIC_SOURCE)
    try:
        text = open(path).read()
        val = float(re.search(r"^traffic_bytes_per_launch:\s*([0-9.eE+]+)", text, re.M).group(1))
        commit = re.search(r"^commit:\s*(\S+)", text, re.M).group(1)
        return val, f"{NCU_TRAFFIC_SOURCE} (ncu --set full at commit {commit})"
    except Exception:
        return None, f"{NCU_TRAFFIC_SOURCE} missing or unreadable"


def schur_bytes(nrhs: int, v5: int, ls: int, real: int = 4) -> float:
    """Algorithmic bytes of one M_pc apply: 120R + 288R/(Ls nrhs) per EVEN 5D site per rhs."""
    return (v5 // 2) * nrhs * (120.0 * real + 288.0 * real / (ls * nrhs))


def apply_bytes(nrhs: int, real: int = 4) -> float:
    """Algorithmic bytes of one D_hop/D_DW/H_DW/D_PV apply: 48R + 72R/(Ls nrhs) per 5D site per rhs."""
    return V5 * nrhs * (48.0 * real + 72.0 * real / (LS * nrhs))


def cheb_bytes(order: int, nvec: int, real: int = 4) -> float:
    """Per order step per 5D site per vector: 6 passes x 24R + 2 gauge reads (D.3)."""
    return order * (V5 * nvec * 144.0 * real + 2 * (V5 // LS) * 72.0 * real)


class ClockSampler:
    """nvidia-smi clocks / throttle reasons during the timed region (B200_PROFILING.md)."""
    Q = ("clocks.sm,clocks.max.sm,clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,"
         "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")

    def __init__(self, index: int):
        self.rows, self.proc = [], None
        try:
            self.proc = subprocess.Popen(["nvidia-smi", f"--id={index}", f"--query-gpu={self.Q}", "--format=csv,noheader,nounits", "-lms", "100"],
                                         stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            self.t = threading.Thread(target=self._read, daemon=True)
            self.t.start()
        except Exception:
            self.proc = None

    def _read(self):
        for line in self.proc.stdout:
            self.rows.append(line.strip())

    def stop(self):
        if self.proc is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        self.proc.terminate()
        try:
            self.proc.wait(timeout=2)
        except Exception:
            self.proc.kill()
        sm, mx, reasons = [], [], set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for r in self.rows:
            p = [v.strip() for v in r.split(",")]
            if len(p) < 6:
                continue
            try:
                sm.append(float(p[0])); mx.append(float(p[1]))
            except ValueError:
                continue
            for n, v in zip(names, p[2:6]):
                if v.lower().startswith("active"):
                    reasons.add(n)
        return {"sm_mhz": statistics.median(sm) if sm else None, "sm_max_mhz": max(mx) if mx else None,
                "reasons": sorted(reasons), "samples": len(sm)}


def oracle_sample(steps: int):
    """The CPU oracle as it stands on the host cores: `steps` fp64 D_DW applies, nrhs = 1, full volume."""
    import numpy as np
    import dwf_inputs as gen
    from oracle import dwf_oracle as oracle
    oracle.build()
    U = gen.gauge_random(L, 1002)
    psi = gen.spinor_gaussian(L, LS, 1, 2002)
    oracle.ddw(U, psi[:, :2], M5, MASS)                      # warm the library / OpenMP pool on a thin slice
    times = []
    for _ in range(steps):
        t0 = time.perf_counter()
        out = oracle.ddw(U, psi, M5, MASS)
        times.append(time.perf_counter() - t0)
        psi = out / np.sqrt(np.mean(np.abs(out) ** 2))
    cores = int(os.environ.get("OMP_NUM_THREADS", os.cpu_count() or 1))
    return times, cores


def oracle_leg(name: str):
    """One D.5 leg of the oracle, run in this (sub)process under whatever OMP_NUM_THREADS it was started with.  Prints a JSON line."""
    import numpy as np
    import dwf_inputs as gen
    from oracle import dwf_oracle as oracle
    oracle.build()
    threads = int(os.environ.get("OMP_NUM_THREADS", os.cpu_count() or 1))
    if name == "ddw":                                        # (i) one fp64 D_DW apply, nrhs = 1, full 16^3x32x16 volume
        U = gen.gauge_random(L, 1002); psi = gen.spinor_gaussian(L, LS, 1, 2002)
        oracle.ddw(U, psi[:, :2], M5, MASS)
        n = 3 if threads > 1 else 1
        t0 = time.perf_counter()
        for _ in range(n):
            oracle.ddw(U, psi, M5, MASS)
        dt = (time.perf_counter() - t0) / n
        out = {"leg": "ddw", "threads": threads, "s_per_apply": round(dt, 3), "GFlop/s": round(FLOP_PER_SITE * V5 / dt / 1e9, 3),
               "sample": f"{n} fp64 D_DW applies, nrhs=1, full 16^3x32x16 volume"}
    elif name == "chebyshev":                                # (ii) Chebyshev of H_DW^2 on ONE vector of the 16^3x32x16 volume
        order = CHEB_ORDER if threads > 1 else 2             # 2*order applies; the single-thread leg is a bounded sample, scaled
        U = gen.gauge_random(L, 1002); psi = gen.spinor_gaussian(L, LS, 1, 2003)
        oracle.ddw(U, psi[:, :2], M5, MASS)
        t0 = time.perf_counter()
        oracle.chebyshev(U, psi, M5, MASS, order, CHEB_LO, CHEB_HI)
        dt = time.perf_counter() - t0
        per_vec = dt * CHEB_ORDER / order
        out = {"leg": "chebyshev", "threads": threads, "order_run": order, "s": round(dt, 2),
               "s_per_order64_vector": round(per_vec, 2), "vectors/s": round(1.0 / per_vec, 5),
               "sample": f"order-{order} filter of 1 vector (2x{order} operator applies), full 16^3x32x16 volume"
                         + ("" if order == CHEB_ORDER else f", scaled x{CHEB_ORDER // order} to order {CHEB_ORDER}")}
    elif name == "cg":                                       # (iii) 10 red-black CG iterations at configs[1] (8^4 x 16)
        L8 = (8, 8, 8, 8)
        U = gen.gauge_random(L8, 1001)
        b = gen.keep_parity(gen.spinor_gaussian(L8, LS, 1, 2001), L8, 0)
        oracle.cg_schur(U, b, M5, MASS, 1)
        t0 = time.perf_counter()
        oracle.cg_schur(U, b, M5, MASS, 10)
        dt = time.perf_counter() - t0
        out = {"leg": "cg", "threads": threads, "s": round(dt, 3), "iterations/s": round(11 / dt, 3),
               "sample": "10 rb-CG iterations (+ the initial residual), 8^4x16, fp64"}
    else:
        raise SystemExit(f"unknown oracle leg {name}")
    print(json.dumps(out), flush=True)


def oracle_legs():
    """the oracle, as it stands, on the host cores: legs (i) D_DW apply, (ii) order-64 Chebyshev on 1 vector,
    (iii) 10 CG iterations at configs[1], each at OMP_NUM_THREADS = 1 and = nproc (subprocesses: OpenMP reads it at start-up)."""
    res = {}
    nproc = os.cpu_count() or 1
    for leg in ("ddw", "chebyshev", "cg"):
        for threads in (nproc, 1):
            env = dict(os.environ, OMP_NUM_THREADS=str(threads))
            try:
                p = subprocess.run([sys.executable, os.path.abspath(__file__), "--oracle-leg", leg], env=env, capture_output=True,
                                   text=True, timeout=600)
                line = [ln for ln in p.stdout.splitlines() if ln.startswith("{")][-1]
                res[f"{leg}_threads{threads}"] = json.loads(line)
            except Exception as exc:                          # a leg that fails must not take the bench line with it
                res[f"{leg}_threads{threads}"] = {"error": repr(exc)[:200]}
    return res


def oracle_mixed_step(state):
    """One reference step = a bounded sample of the bench step's own mix, on the full 16^3x32x16 volume, one right-hand side, fp64:
    a2-a4 D_hop, D_DW, H_DW, D_PV (4 applies) | a5/a6 M_pc (1) | a7 axpy/inner/norm2 | a8 Chebyshev of order 1 (2) |
    a9 one rb-CG iteration incl. the initial residual at configs[1]'s 8^4 x 16 (4 applies of 1/32 of the volume).
    Returns (seconds, D_DW-equivalent applies of the 16^3x32x16 volume)."""
    import numpy as np
    import dwf_inputs as gen
    from oracle import dwf_oracle as oracle
    if not state:
        oracle.build()
        state["U"] = gen.gauge_random(L, 1002)
        state["psi"] = gen.spinor_gaussian(L, LS, 1, 2002)
        state["psi_e"] = gen.keep_parity(state["psi"], L, 0)
        state["U8"] = gen.gauge_random((8, 8, 8, 8), 1001)
        state["b8"] = gen.keep_parity(gen.spinor_gaussian((8, 8, 8, 8), LS, 1, 2001), (8, 8, 8, 8), 0)
        oracle.ddw(state["U"], state["psi"][:, :2], M5, MASS)   # warm the library / OpenMP pool on a thin slice
    U, psi, pe = state["U"], state["psi"], state["psi_e"]
    t0 = time.perf_counter()
    oracle.dhop(U, psi); y = oracle.ddw(U, psi, M5, MASS); oracle.hdw(U, psi, M5, MASS); oracle.dpv(U, psi, M5)
    oracle.mpc(U, pe, M5, MASS)
    oracle.axpy([0.5 + 0.1j], psi, y); oracle.inner(psi, y); oracle.norm2(psi)
    oracle.chebyshev(U, psi, M5, MASS, 1, CHEB_LO, CHEB_HI)
    oracle.cg_schur(state["U8"], state["b8"], M5, MASS, 1)
    return time.perf_counter() - t0, 4 + 1 + 2 + 4 * (8 ** 4) / (L[0] * L[1] * L[2] * L[3])


def run_reference(args):
    """--impl reference: the oracle timed on the host cores (this tier's reference arm)."""
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    state = {}
    for _ in range(min(args.warmup, 1)):
        oracle_mixed_step(state)
    times, applies = [], 0
    for _ in range(args.steps):
        dt, n = oracle_mixed_step(state)
        times.append(dt); applies += n
    total = sum(times)
    cores = int(os.environ.get("OMP_NUM_THREADS", os.cpu_count() or 1))
    val = FLOP_PER_SITE * V5 * applies / total / 1e9
    sample = ("per step, on the full 16^3x32x16 volume, one rhs, fp64: D_hop, D_DW, H_DW, D_PV, M_pc, axpy/inner/norm2, order-1 Chebyshev, "
              "one rb-CG iteration at 8^4x16 (7.1 D_DW-equivalent applies: a bounded sample of every row of the bench step)")
    line = {"impl": "reference", "metric": "D_DW-equivalent GFlop/s @1320 flop per 5D site", "value": val, "unit": "GFlop/s",
            "n_gpus": args.gpus, "steps": args.steps, "warmup": args.warmup, "ms_per_step": 1e3 * total / max(args.steps, 1),
            "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": {"workload": WORKLOAD, "sample": sample},
            "cpu_baseline": {"value": val, "unit": "GFlop/s", "cores": cores, "kind": "oracle", "sample": f"{args.steps} steps; " + sample},
            "e2e": {"value": val, "unit": "GFlop/s", "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0}
    print(json.dumps(line), flush=True)


def combine_over_ranks(ms: float, launches: int, dev, world: int):
    """Replicas: the job's time is the MAX over ranks, its kernel-launch count the SUM."""
    if world <= 1:
        return ms, launches
    import torch
    import torch.distributed as dist
    tt = torch.tensor([ms], device=dev, dtype=torch.float64)
    dist.all_reduce(tt, op=dist.ReduceOp.MAX)
    ll = torch.tensor([launches], device=dev, dtype=torch.int64)
    dist.all_reduce(ll)
    return float(tt.item()), int(ll.item())


def run_only(args, dev):
    """Time a single part of the step (used for ncu captures and kernel tuning)."""
    import torch

    import dwf_inputs as gen
    from paper_2103_05034_b200 import DWF_DDW, DWF_DHOP, DWF_F32, DWF_F64, DWF_HDW, DWF_SCHUR_EO, Dwf
    f32 = args.prec == "f32"
    name = args.only
    if name.endswith("_48"):
        return run_only_config4(args, dev)
    if name == "subspace":                                   # eq. 34-37 on 16^3x32x16 fp32, one noise vector
        m, lam_lo, lam_max, delta, nvec = 64, 0.5, 60.0, 16, 5
        d = Dwf(L, LS, M5, MASS, DWF_F32, device=dev)
        d.set_gauge(torch.from_numpy(gen.gauge_random(L, 1002)).to(d.cdtype).to(dev))
        d.set_workspace(1)
        g = torch.Generator(device=dev); g.manual_seed(2007)
        eta = d.field(1).normal_(generator=g)
        phi = torch.empty(nvec * eta.numel(), dtype=d.rdtype, device=dev)
        lam, _ = d.power_lambda_max(20, eta.clone())
        for _ in range(3):
            d.chebyshev_subspace(m, lam_lo, lam_max, delta, nvec, eta, phi, 1)
        torch.cuda.synchronize()
        a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        a.record()
        for _ in range(args.steps):
            d.chebyshev_subspace(m, lam_lo, lam_max, delta, nvec, eta, phi, 1)
        b.record(); torch.cuda.synchronize()
        ms = a.elapsed_time(b) / args.steps
        applies = 2 * m + 2 * (nvec - 1) * delta
        print(json.dumps({"only": name, "m": m, "delta": delta, "nvec": nvec, "lambda_max_power20": round(lam, 3), "ms": round(ms, 3),
                          "H_applies": applies, "us_per_apply": round(1e3 * ms / applies, 1), "vectors/s": round(nvec / ms * 1e3, 1),
                          "GFlop/s": round(FLOP_PER_SITE * V5 * applies / ms / 1e6, 1)}), flush=True)
        return
    if name == "solve":                                      # complete red-black solve of D_DW psi = eta to 1e-8 (fp32 + mixed)
        d = Dwf(L, LS, M5, MASS, DWF_F32, device=dev)
        U = gen.gauge_random(L, 1002)
        d.set_gauge(torch.from_numpy(U).to(d.cdtype).to(dev))
        d.set_workspace(1)
        g = torch.Generator(device=dev); g.manual_seed(2011)
        eta = d.field(1).normal_(generator=g); psi = d.field(1)
        d.solve(eta, psi, 1e-5, 4000)
        torch.cuda.synchronize(); t0 = time.perf_counter()
        iters, relres = d.solve(eta, psi, 1e-5, 4000)
        torch.cuda.synchronize(); ms32 = (time.perf_counter() - t0) * 1e3
        d64 = Dwf(L, LS, M5, MASS, DWF_F64, device=dev)
        d64.set_gauge(torch.from_numpy(U).to(d64.cdtype).to(dev))
        d64.set_workspace(1)
        eta64 = d.convert_to(d64, eta, 1); psi64 = d64.field(1)
        d64.solve_mixed(d, eta64, psi64, 1e-10, 1e-4, 20, 4000)
        torch.cuda.synchronize(); t0 = time.perf_counter()
        outer, inner, rr = d64.solve_mixed(d, eta64, psi64, 1e-10, 1e-4, 20, 4000)
        torch.cuda.synchronize(); msmx = (time.perf_counter() - t0) * 1e3
        torch.cuda.synchronize(); t0 = time.perf_counter()
        it64, rr64 = d64.solve(eta64, psi64, 1e-10, 4000)
        torch.cuda.synchronize(); ms64 = (time.perf_counter() - t0) * 1e3
        print(json.dumps({"only": name, "fp32_tol1e-5": {"iters": iters, "relres": relres, "ms": round(ms32, 2)},
                          "mixed_tol1e-10": {"outer": outer, "inner_iters": inner, "relres": rr, "ms": round(msmx, 2)},
                          "fp64_tol1e-10": {"iters": it64, "relres": rr64, "ms": round(ms64, 2)}}), flush=True)
        return
    if name == "cg_8":                                       # BASELINE.json configs[1]: 8^4 x 16, 50 rb-CG iterations (launch-bound size)
        L8 = (8, 8, 8, 8)
        d = Dwf(L8, LS, M5, MASS, DWF_F32 if f32 else DWF_F64, device=dev)
        d.set_gauge(torch.from_numpy(gen.gauge_random(L8, 1001)).to(d.cdtype).to(dev))
        d.set_workspace(1)
        g = torch.Generator(device=dev); g.manual_seed(2001)
        b = d.field(1, half=True).normal_(generator=g); x = d.field(1, half=True, zero=True)
        for _ in range(3):
            x.zero_(); d.cg_schur(b, x, 50)
        torch.cuda.synchronize()
        t0 = time.perf_counter()
        for _ in range(args.steps):
            x.zero_(); d.cg_schur(b, x, 50)
        torch.cuda.synchronize()
        ms = (time.perf_counter() - t0) * 1e3 / args.steps
        print(json.dumps({"only": name, "prec": args.prec, "iters": 50, "ms": round(ms, 3), "iterations/s": round(51 / ms * 1e3, 1)}), flush=True)
        return
    if name == "blas1":                                      # a7 on 12 full fields: axpy, inner, norm2
        d = Dwf(L, LS, M5, MASS, DWF_F32 if f32 else DWF_F64, device=dev)
        g = torch.Generator(device=dev); g.manual_seed(2002)
        x, y = d.field(12).normal_(generator=g), d.field(12).normal_(generator=g)
        ms = time_calls(lambda j: (d.axpy([0.5 + 0.1j] * 12, x, y, 12), d.inner(x, y, 12), d.norm2(x, 12)), args.steps)
        by = 144.0 * (4 if f32 else 8) * V5 * 12
        print(json.dumps({"only": name, "prec": args.prec, "nrhs": 12, "ms": round(ms, 4), "GB/s": round(by / ms / 1e6, 1),
                          "frac_of_hbm_peak": round(by / ms / 1e6 / peaks()[0], 4)}), flush=True)
        return
    d = Dwf(L, LS, M5, MASS, DWF_F32 if f32 else DWF_F64, device=dev)
    d.set_gauge(torch.from_numpy(gen.gauge_random(L, 1002)).to(d.cdtype).to(dev))
    g = torch.Generator(device=dev); g.manual_seed(2002)
    nrhs = int(name.split("nrhs")[1]) if "nrhs" in name else (CHEB_NVEC if name == "chebyshev" else 1)
    d.set_workspace(nrhs)
    half = name.startswith("schur") or name == "cg"
    nb = 4 if nrhs == 1 else 1
    xs = [d.field(nrhs, half=half).normal_(generator=g) for _ in range(nb)]
    ys = [d.field(nrhs, half=half) for _ in range(nb)]
    ops = {"dhop": DWF_DHOP, "ddw": DWF_DDW, "hdw": DWF_HDW, "schur": DWF_SCHUR_EO}

    def once(j):
        if name == "chebyshev":
            d.chebyshev(CHEB_ORDER, CHEB_LO, CHEB_HI, xs[0], ys[0], nrhs)
        elif name == "cg":
            ys[0].zero_(); d.cg_schur(xs[0], ys[0], CG_ITERS)
        else:
            d.apply(ops[name.split("_")[0]], xs[j % nb], ys[j % nb], nrhs)
    for j in range(max(args.warmup, 3)):
        once(j)
    torch.cuda.synchronize()
    a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    a.record()
    for j in range(args.steps):
        once(j)
    b.record(); torch.cuda.synchronize()
    ms = a.elapsed_time(b) / args.steps
    out = {"only": name, "prec": args.prec, "nrhs": nrhs, "ms": round(ms, 4)}
    if name.split("_")[0] in ("dhop", "ddw", "hdw"):
        by = apply_bytes(nrhs, 4 if f32 else 8)
        out.update({"GB/s": round(by / ms / 1e6, 1), "GFlop/s": round(FLOP_PER_SITE * V5 * nrhs / ms / 1e6, 1),
                    "frac_of_hbm_peak": round(by / ms / 1e6 / peaks()[0], 4)})
    print(json.dumps(out), flush=True)


def run_only_config4(args, dev):
    """BASELINE.json configs[4]: 48^3 x 96 x Ls=24 fp32, m = 0.00078: one D_DW apply / 100 rb-CG iterations."""
    import torch

    import dwf_inputs as gen
    from paper_2103_05034_b200 import DWF_DDW, DWF_F32, Dwf
    L4, LS4, MASS4 = (48, 48, 48, 96), 24, 0.00078
    v5 = L4[0] * L4[1] * L4[2] * L4[3] * LS4
    d = Dwf(L4, LS4, M5, MASS4, DWF_F32, device=dev)
    d.set_gauge(gen.gauge_random_torch(L4, 1004, dev, torch.complex64))
    g = torch.Generator(device=dev); g.manual_seed(2004)
    a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    if args.only == "ddw_48":
        x, y = d.field(1).normal_(generator=g), d.field(1)
        for _ in range(max(args.warmup, 3)):
            d.apply(DWF_DDW, x, y, 1)
        a.record()
        for _ in range(args.steps):
            d.apply(DWF_DDW, x, y, 1)
        b.record(); torch.cuda.synchronize()
        ms = a.elapsed_time(b) / args.steps
        by = v5 * (48.0 * 4 + 72.0 * 4 / LS4)
        out = {"only": "ddw_48", "ms": round(ms, 3), "GB/s": round(by / ms / 1e6, 1), "GFlop/s": round(FLOP_PER_SITE * v5 / ms / 1e6, 1),
               "frac_of_hbm_peak": round(by / ms / 1e6 / peaks()[0], 4)}
    else:
        d.set_workspace(1, half_fields=5)
        bb, xx = d.field(1, half=True).normal_(generator=g), d.field(1, half=True, zero=True)
        d.cg_schur(bb, xx, 3)
        xx.zero_(); torch.cuda.synchronize()
        a.record(); hist = d.cg_schur(bb, xx, 100); b.record(); torch.cuda.synchronize()
        ms = a.elapsed_time(b)
        out = {"only": "cg_48", "iters": 100, "ms": round(ms, 2), "iterations/s": round(101 / ms * 1e3, 2),
               "resid2_first_last": [hist[0], hist[-1]]}
    print(json.dumps(out), flush=True)


def time_calls(fn, n, warm=3):
    """Average milliseconds of fn(j) over n back-to-back calls (CUDA events on the current stream)."""
    import torch
    for j in range(warm):
        fn(j)
    torch.cuda.synchronize()
    a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    a.record()
    for j in range(n):
        fn(j)
    b.record(); torch.cuda.synchronize()
    return a.elapsed_time(b) / n


def run_extras(dev, peak):
    """Numbers of BASELINE.md that are not part of the timed fp32 step (SURVEY 8(d) D.1 rows [1], [2] fp64, [4]): run once,
    after the step's buffers are freed.  Returns a dict for `detail`."""
    import gc
    import torch
    import dwf_inputs as gen
    from paper_2103_05034_b200 import DWF_DDW, DWF_F32, DWF_F64, DWF_HDW, DWF_SCHUR_EO, Dwf
    out = {}
    # ---- configs[2] in fp64 (the paper's own precision): D_DW and H_DW at nrhs 1 / 12 / 48
    d = Dwf(L, LS, M5, MASS, DWF_F64, device=dev)
    d.set_gauge(torch.from_numpy(gen.gauge_random(L, 1002)).to(torch.complex128).to(dev))
    g = torch.Generator(device=dev); g.manual_seed(2002)
    for nrhs, reps in ((1, 20), (12, 3), (48, 2)):
        nb = 4 if nrhs == 1 else 1
        xs = [d.field(nrhs).normal_(generator=g) for _ in range(nb)]
        ys = [d.field(nrhs) for _ in range(nb)]
        for name, op in (("ddw", DWF_DDW), ("hdw", DWF_HDW)):
            ms = time_calls(lambda j: d.apply(op, xs[j % nb], ys[j % nb], nrhs), reps, warm=2)
            by = apply_bytes(nrhs, 8)
            out[f"{name}_nrhs{nrhs}_fp64"] = {"ms": round(ms, 4), "GB/s": round(by / ms / 1e6, 1), "GFlop/s": round(FLOP_PER_SITE * V5 * nrhs / ms / 1e6, 1),
                                             "frac_of_hbm_peak": round(by / ms / 1e6 / peak, 4)}
        del xs, ys
    d.set_workspace(4, half_fields=1)
    xs4 = d.field(4, half=True).normal_(generator=g); ys4 = d.field(4, half=True)
    ms = time_calls(lambda j: d.apply(DWF_SCHUR_EO, xs4, ys4, 4), 5)
    by = schur_bytes(4, V5, LS, 8)
    out["schur_nrhs4_fp64"] = {"ms": round(ms, 4), "GB/s": round(by / ms / 1e6, 1), "frac_of_hbm_peak": round(by / ms / 1e6 / peak, 4)}
    del xs4, ys4
    d.close(); del d
    gc.collect(); torch.cuda.empty_cache()
    # ---- Table V rows 1-2 on the synthetic 16^3x32x16 field (fp32): unpreconditioned CGNR on M^dag M and BiCGSTAB on M_PV^dag M,
    # 20 iterations each, iterations/s and the number of full-lattice operator applies per iteration (2 and 4)
    d = Dwf(L, LS, M5, MASS, DWF_F32, device=dev)
    d.set_gauge(torch.from_numpy(gen.gauge_random(L, 1002)).to(torch.complex64).to(dev))
    d.set_workspace(1)
    g = torch.Generator(device=dev); g.manual_seed(2012)
    bfull = d.field(1).normal_(generator=g); xfull = d.field(1, zero=True)
    for name, fn, applies in (("cgnr_MdagM", lambda: d.cg_normal(bfull, xfull.zero_(), 20, 1), 2),
                              ("bicgstab_MpvdagM", lambda: d.bicgstab_pv(bfull, xfull.zero_(), 20), 4)):
        fn(); torch.cuda.synchronize(); t0 = time.perf_counter()
        for _ in range(3):
            fn()
        torch.cuda.synchronize()
        ms = (time.perf_counter() - t0) * 1e3 / 3
        out[f"{name}_16^3x32x16_fp32"] = {"iters": 20, "ms": round(ms, 3), "iterations/s": round(21 / ms * 1e3, 1),
                                          "full_applies_per_iteration": applies,
                                          "GFlop/s": round(FLOP_PER_SITE * V5 * applies * 21 / ms / 1e6, 1)}
    d.close(); del d, bfull, xfull
    gc.collect(); torch.cuda.empty_cache()
    # ---- configs[1]: 8^4 x 16, 50 rb-CG iterations (launch-bound size), fp32 and fp64
    L8 = (8, 8, 8, 8)
    for prec, code, cdt in (("fp32", DWF_F32, torch.complex64), ("fp64", DWF_F64, torch.complex128)):
        d = Dwf(L8, LS, M5, MASS, code, device=dev)
        d.set_gauge(torch.from_numpy(gen.gauge_random(L8, 1001)).to(cdt).to(dev))
        d.set_workspace(1, half_fields=5)
        g = torch.Generator(device=dev); g.manual_seed(2001)
        b = d.field(1, half=True).normal_(generator=g); x = d.field(1, half=True, zero=True)

        def cg50(j):
            x.zero_(); d.cg_schur(b, x, 50)
        for _ in range(3):
            cg50(0)
        torch.cuda.synchronize(); t0 = time.perf_counter()
        for j in range(10):
            cg50(j)
        torch.cuda.synchronize()
        ms = (time.perf_counter() - t0) * 1e3 / 10             # host clock: the call synchronises and is launch-bound
        out[f"rb_cg_8^4x16_{prec}"] = {"iters": 50, "ms": round(ms, 3), "iterations/s": round(51 / ms * 1e3, 1)}
        d.close(); del d, b, x
    gc.collect(); torch.cuda.empty_cache()
    # ---- configs[4]: 48^3 x 96 x 24 fp32, m = 0.00078: one D_DW apply, the Schur operator, 100 rb-CG iterations
    free, _ = torch.cuda.mem_get_info()
    if free < 120e9:
        out["config4"] = {"skipped": f"needs ~110 GB of device memory, {free / 1e9:.0f} GB free"}
        return out
    L4, LS4, MASS4 = (48, 48, 48, 96), 24, 0.00078
    v5 = L4[0] * L4[1] * L4[2] * L4[3] * LS4
    d = Dwf(L4, LS4, M5, MASS4, DWF_F32, device=dev)
    d.set_gauge(gen.gauge_random_torch(L4, 1004, dev, torch.complex64))
    g = torch.Generator(device=dev); g.manual_seed(2004)
    x, y = d.field(1).normal_(generator=g), d.field(1)
    ms = time_calls(lambda j: d.apply(DWF_DDW, x, y, 1), 5, warm=2)
    by = v5 * (48.0 * 4 + 72.0 * 4 / LS4)
    out["ddw_48^3x96x24_fp32"] = {"ms": round(ms, 3), "GB/s": round(by / ms / 1e6, 1), "GFlop/s": round(FLOP_PER_SITE * v5 / ms / 1e6, 1),
                                  "frac_of_hbm_peak": round(by / ms / 1e6 / peak, 4)}
    del y
    d.set_workspace(1, half_fields=5)
    hb = d.field_bytes(1, half=True) // 4
    bb = x[:hb].clone(); del x
    xx = d.field(1, half=True, zero=True)
    ms = time_calls(lambda j: d.apply(DWF_SCHUR_EO, bb, xx, 1), 3, warm=1)
    by = schur_bytes(1, v5, LS4, 4)
    out["schur_48^3x96x24_fp32"] = {"ms": round(ms, 3), "GB/s": round(by / ms / 1e6, 1), "frac_of_hbm_peak": round(by / ms / 1e6 / peak, 4)}
    d.cg_schur(bb, xx, 2)
    xx.zero_(); torch.cuda.synchronize()
    a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    a.record(); hist = d.cg_schur(bb, xx, 100); b.record(); torch.cuda.synchronize()
    ms = a.elapsed_time(b)
    out["rb_cg_48^3x96x24_fp32"] = {"iters": 100, "ms": round(ms, 1), "iterations/s": round(101 / ms * 1e3, 2),
                                    "resid2_first_last": [hist[0], hist[-1]]}
    d.close(); del d, bb, xx
    gc.collect(); torch.cuda.empty_cache()
    return out


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=3)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="dwf", choices=["dwf", "reference"])
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--only", default=None, help="time one part of the step only (for ncu captures), e.g. ddw_nrhs1, "
                    "hdw_nrhs1, dhop_nrhs1, ddw_nrhs12, ddw_nrhs48, schur_nrhs4, chebyshev, cg, cg_8, blas1, ddw_48, cg_48, subspace, solve; prints a small JSON line")
    ap.add_argument("--prec", default="f32", choices=["f32", "f64"], help="--only mode: precision")
    ap.add_argument("--no-extras", action="store_true", help="skip the fp64 / 8^4 / 48^3x96 legs of `detail` (run once, outside the timed step)")
    ap.add_argument("--oracle-leg", default=None, help=argparse.SUPPRESS)
    args = ap.parse_args()
    if args.oracle_leg:
        return oracle_leg(args.oracle_leg)
    if args.impl == "reference":
        return run_reference(args)

    import torch
    import torch.distributed as dist

    import dwf_inputs as gen
    from paper_2103_05034_b200 import (DWF_DDW, DWF_DHOP, DWF_DPV, DWF_F32, DWF_HDW, DWF_SCHUR_EO, Dwf)

    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device(f"cuda:{local}"))
    dev = torch.device(f"cuda:{local}")
    torch.cuda.set_device(dev)
    warmup = max(args.warmup, 3)
    if args.only:
        return run_only(args, dev)

    # ---- inputs (seeded, synthetic): SU(3) links from dwf_inputs (host), spinors iid N(0,1)
    # drawn directly in the native layout by torch's seeded CUDA generator (a permutation of iid Gaussians).
    d = Dwf(L, LS, M5, MASS, DWF_F32, device=dev)
    U = torch.from_numpy(gen.gauge_random(L, 1002)).to(torch.complex64).to(dev)
    d.set_gauge(U)
    del U
    d.set_workspace(CHEB_NVEC)
    g = torch.Generator(device=dev); g.manual_seed(2002 + rank)

    def rnd(nrhs, half=False):
        f = d.field(nrhs, half=half)
        f.normal_(generator=g)
        return f

    NB = 4                                                   # rotate buffers so nrhs=1 applies stream from HBM
    x1 = [rnd(1) for _ in range(NB)]; y1 = [d.field(1) for _ in range(NB)]
    x12, y12 = rnd(12), d.field(12)
    x48, y48 = rnd(48), d.field(48)
    xs4, ys4 = rnd(4, half=True), d.field(4, half=True)
    xc, yc = rnd(CHEB_NVEC), d.field(CHEB_NVEC)
    bcg, xcg = rnd(1, half=True), d.field(1, half=True)
    canon = torch.randn(d.canonical_shape(1) + (2,), generator=g, device=dev, dtype=torch.float32)
    canon = torch.view_as_complex(canon).contiguous()
    host_in = torch.empty(d.canonical_shape(1), dtype=torch.complex64).pin_memory()
    host_in.copy_(canon.cpu())
    host_out = torch.empty_like(host_in).pin_memory()

    ev = lambda: torch.cuda.Event(enable_timing=True)
    parts = {}

    def timed(name, fn):
        a, b = ev(), ev()
        a.record(); fn(); b.record()
        parts.setdefault(name, []).append((a, b))

    hop_applies = {"n": 0.0}

    def step(record):
        t = timed if record else (lambda name, fn: fn())
        hop = 0.0
        t("a1_import_export", lambda: d.export(d.import_(canon, x1[0]), 1, canonical=canon))
        for i, op in enumerate((DWF_DHOP, DWF_DDW, DWF_HDW, DWF_DPV)):
            name = ("dhop", "ddw", "hdw", "dpv")[i] + "_nrhs1"
            for j in range(NB):
                t(name, lambda: d.apply(op, x1[j], y1[j], 1))
            hop += NB
        t("ddw_nrhs12", lambda: d.apply(DWF_DDW, x12, y12, 12)); hop += 12
        t("ddw_nrhs48", lambda: d.apply(DWF_DDW, x48, y48, 48)); hop += 48
        t("schur_nrhs4", lambda: d.apply(DWF_SCHUR_EO, xs4, ys4, 4)); hop += 4
        t("blas1_nrhs12", lambda: (d.axpy([0.5 + 0.1j] * 12, x12, y12, 12), d.inner(x12, y12, 12), d.norm2(x12, 12)))
        t("chebyshev", lambda: d.chebyshev(CHEB_ORDER, CHEB_LO, CHEB_HI, xc, yc, CHEB_NVEC)); hop += 2 * CHEB_ORDER * CHEB_NVEC
        xcg.zero_()
        t("cg", lambda: d.cg_schur(bcg, xcg, CG_ITERS)); hop += 2 * (CG_ITERS + 1)
        hop_applies["n"] = hop

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    for _ in range(warmup):
        step(False)
    barrier()
    sampler = ClockSampler(local) if rank == 0 else None
    l0 = d.launch_count()
    s, e = ev(), ev()
    s.record()
    for _ in range(args.steps):
        step(True)
    e.record()
    barrier()
    clocks = sampler.stop() if sampler else None
    launches = d.launch_count() - l0
    ms = s.elapsed_time(e)
    ms, launches = combine_over_ranks(ms, launches, dev, world)

    # ---- e2e: the same apply through the C ABI with HOST buffers (H2D + D2H inside the timed region)
    for _ in range(2):
        d.apply_host(DWF_DDW, host_in, host_out, 1)
    barrier()
    t0 = time.perf_counter()
    ne2e = 3
    for _ in range(ne2e):
        d.apply_host(DWF_DDW, host_in, host_out, 1)
    torch.cuda.synchronize()
    e2e_s = (time.perf_counter() - t0) / ne2e
    e2e_s, _ = combine_over_ranks(e2e_s, 0, dev, world)

    if rank != 0:
        if world > 1:
            dist.destroy_process_group()
        return

    def avg_ms(name):
        v = [a.elapsed_time(b) for a, b in parts[name]]
        return sum(v) / len(v)

    peak, peak_src = peaks()
    detail = {}
    for name, nrhs in (("dhop_nrhs1", 1), ("ddw_nrhs1", 1), ("hdw_nrhs1", 1), ("dpv_nrhs1", 1), ("ddw_nrhs12", 12), ("ddw_nrhs48", 48)):
        t_ms = avg_ms(name)
        detail[name] = {"ms": round(t_ms, 4), "GB/s": round(apply_bytes(nrhs) / t_ms / 1e6, 1),
                        "GFlop/s": round(FLOP_PER_SITE * V5 * nrhs / t_ms / 1e6, 1),
                        "frac_of_hbm_peak": round(apply_bytes(nrhs) / t_ms / 1e6 / peak, 4)}
    t_cheb = avg_ms("chebyshev")
    detail["chebyshev_order64_24vec"] = {"ms": round(t_cheb, 3), "vectors/s": round(CHEB_NVEC / t_cheb * 1e3, 2),
                                          "GB/s": round(cheb_bytes(CHEB_ORDER, CHEB_NVEC) / t_cheb / 1e6, 1)}
    t_cg = avg_ms("cg")
    detail["rb_cg_16^3x32x16"] = {"ms": round(t_cg, 3), "iterations/s": round((CG_ITERS + 1) / t_cg * 1e3, 1)}
    detail["a1_import_export"] = {"ms": round(avg_ms("a1_import_export"), 4),
                                  "GB/s": round(2 * 48.0 * 4 * V5 / avg_ms("a1_import_export") / 1e6, 1)}      # import + export: 2 x (R + W)
    t_s = avg_ms("schur_nrhs4")
    detail["schur_nrhs4"] = {"ms": round(t_s, 4), "GB/s": round(schur_bytes(4, V5, LS) / t_s / 1e6, 1),
                             "frac_of_hbm_peak": round(schur_bytes(4, V5, LS) / t_s / 1e6 / peak, 4),
                             "GFlop/s": round(FLOP_PER_SITE * V5 * 4 / t_s / 1e6, 1)}
    t_b = avg_ms("blas1_nrhs12")
    blas_bytes = (72.0 + 48.0 + 24.0) * 4 * V5 * 12                                   # axpy 72R + inner 48R + norm 24R per 5D site per rhs
    detail["blas1_nrhs12"] = {"ms": round(t_b, 4), "GB/s": round(blas_bytes / t_b / 1e6, 1), "frac_of_hbm_peak": round(blas_bytes / t_b / 1e6 / peak, 4),
                              "note": "axpy + inner + norm2 on 12 full fields, two host synchronisations inside"}

    # dominant kernel = dwf::hop_tile_kernel inside dwf_chebyshev (H_DW and H_DW + three-term-recurrence epilogues,
    # one launch per right-hand side and apply).  Its average launch duration = CUDA-event-bracketed call time
    # on the launching stream / launches of the call; algorithmic bytes per launch = cheb_bytes / launches.
    lc0 = d.launch_count()
    d.chebyshev(CHEB_ORDER, CHEB_LO, CHEB_HI, xc, yc, CHEB_NVEC)
    torch.cuda.synchronize()
    n_launch = d.launch_count() - lc0
    ach = cheb_bytes(CHEB_ORDER, CHEB_NVEC) / t_cheb / 1e6
    roofline = {"bound": "hbm", "kernel": "dwf::hop_tile_kernel<float,16,32,...> (H_DW and H_DW+axpby epilogues, inside dwf_chebyshev)",
                "achieved": round(ach, 1), "peak": peak, "peak_source": peak_src, "unit": "GB/s", "frac": round(ach / peak, 4),
                "traffic": ncu_traffic()[0], "traffic_source": ncu_traffic()[1],
                "algorithmic_bytes_per_launch": round(cheb_bytes(CHEB_ORDER, CHEB_NVEC) / n_launch),
                "avg_launch_ms": round(t_cheb / n_launch, 4), "launches_per_call": n_launch,
                "co_limit": "packed-fp32 FMA pipe: ~906 FFMA2/FADD2/FMUL2 per 2 5D sites, measured 100 lane-FMA/clk/SM (DESIGN.md sec. 5.2)",
                "ddw_nrhs1_frac": detail["ddw_nrhs1"]["frac_of_hbm_peak"]}

    total_flop = FLOP_PER_SITE * V5 * hop_applies["n"] * args.steps * world
    value = total_flop / ms / 1e6
    e2e_val = FLOP_PER_SITE * V5 * world / e2e_s / 1e9
    fb = d.field_bytes(1)
    line = {"metric": "D_DW-equivalent GFlop/s @1320 flop per 5D site", "value": round(value, 1), "unit": "GFlop/s", "n_gpus": world,
            "steps": args.steps, "warmup": warmup, "ms_per_step": round(ms / args.steps, 3), "higher_is_better": True,
            "scaling": "weak", "vs_baseline": None, "dtype": "f32", "data": "synthetic",
            "config": {"workload": WORKLOAD, "lattice": "16x16x16x32", "Ls": LS, "M5": M5, "mass": MASS,
                       "l2": "inputs larger than L2 (nrhs>=12 fields >= 2.4 GB); nrhs=1 applies rotate over 4 buffer pairs (1.6 GB)",
                       "parallelism": "replicas" if world > 1 else "single GPU"},
            "clocks": clocks, "gpu_launches": int(launches),
            "e2e": {"value": round(e2e_val, 2), "unit": "GFlop/s", "h2d_bytes_per_step": fb, "d2h_bytes_per_step": fb,
                    "call": "dwf_apply_host(DWF_DDW, nrhs=1): pinned host canonical in -> H2D -> import -> D_DW -> export -> D2H, pipelined over 16 chunks of t-slices (both copy directions at once)",
                    "ms": round(e2e_s * 1e3, 3)},
            "roofline": roofline, "detail": detail}
    if not args.no_extras and world == 1:
        # free the step's buffers, then the legs that need their own handles (fp64, 8^4, 48^3 x 96)
        del x1, y1, x12, y12, x48, y48, xs4, ys4, xc, yc, bcg, xcg, canon
        d.close()
        import gc
        gc.collect(); torch.cuda.empty_cache()
        try:
            detail.update(run_extras(dev, peak))
        except Exception as exc:                              # the headline line must survive a failing extra leg
            detail["extras_error"] = repr(exc)[:300]
    if not args.no_cpu_baseline and world == 1:
        line["cpu_baseline_legs"] = oracle_legs()
        times, cores = oracle_sample(5)
        tot = sum(times)
        line["cpu_baseline"] = {"value": round(FLOP_PER_SITE * V5 * len(times) / tot / 1e9, 3), "unit": "GFlop/s", "cores": cores,
                                "kind": "oracle", "sample": "5 fp64 D_DW applies (nrhs=1) on the full 16^3x32x16 volume",
                                "ms_per_apply": round(1e3 * tot / len(times), 1)}
    print(json.dumps(line), flush=True)
    if world > 1:
        dist.destroy_process_group()


if __name__ == "__main__":
    main()
