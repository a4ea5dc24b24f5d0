#!/usr/bin/env python
"""bench.py — whole-hot-path benchmark of libhr_dslash on BASELINE.json configs[3]/[4] (48^4).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference] [--L 48]

One "step" = one pass of every hot-path row of DESIGN.md §2 over one 48^4 lattice of synthetic seeded
fields (Haar links, Gaussian spinors; clover links exp(i 0.3 a.sigma)), inputs resident in HBM:
    fp64: H1 hop o<-e, H1 hop e<-o, H3 full D, E1 Dhat, C2 clover, C3 clover inverse, E2 Dhat+clover, R1 represent
    fp32: H1 hop o<-e, H1 hop e<-o, H3 full D, E1 Dhat
`value` = compulsory (algorithmic) bytes of the step (hr_dirac_flops_bytes) / step time, in GB/s — the paper's
bandwidth metric.  Prints ONE JSON line (rank 0).  See DESIGN.md §7 for every field.
"""
from __future__ import annotations

import argparse
import json
import os
import sys
import threading
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

METRIC = "dslash_hbm_bandwidth_48^4"
UNIT = "GB/s"


def parse():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=30)
    ap.add_argument("--warmup", type=int, default=5)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--L", type=int, default=48, help="lattice extent (48 = BASELINE.json configs[3]; others for debugging)")
    ap.add_argument("--kernel", default="auto", choices=["auto", "generic", "tiled"])
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--no-cpu", action="store_true")
    ap.add_argument("--no-other", action="store_true", help="skip the 16^4 / 24^4 side report")
    return ap.parse_args()


def peaks():
    """roofline denominator: measured copy bandwidth of this pool's B200s (MEASURED_PEAKS.json), else the
    profiling guide's fallback 6650 GB/s"""
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    try:
        with open(p) as f:
            return float(json.load(f)["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs)"
    except Exception:
        return 6650.0, "fallback (B200_PROFILING.md)"


class ClockSampler(threading.Thread):
    """samples SM clock and throttle reasons through NVML (what nvidia-smi reads) while the timed region runs"""

    def __init__(self, device_index, period=0.02):
        super().__init__(daemon=True)
        self.period = period
        self.samples, self.reasons = [], set()
        self.max_mhz = None
        self.stop_flag = threading.Event()
        self.ok = False
        try:
            import pynvml
            import torch
            pynvml.nvmlInit()
            self.nv = pynvml
            h = None
            try:
                uuid = str(torch.cuda.get_device_properties(device_index).uuid)
                if not uuid.startswith("GPU-"):
                    uuid = "GPU-" + uuid
                h = pynvml.nvmlDeviceGetHandleByUUID(uuid.encode() if hasattr(uuid, "encode") else uuid)
            except Exception:
                h = pynvml.nvmlDeviceGetHandleByIndex(device_index)
            self.h = h
            self.max_mhz = float(pynvml.nvmlDeviceGetMaxClockInfo(h, pynvml.NVML_CLOCK_SM))
            self.ok = True
        except Exception as e:  # pragma: no cover
            self.err = repr(e)

    def run(self):
        if not self.ok:
            return
        nv = self.nv
        names = {
            getattr(nv, "nvmlClocksThrottleReasonHwSlowdown", 0x8): "hw_slowdown",
            getattr(nv, "nvmlClocksThrottleReasonHwThermalSlowdown", 0x40): "hw_thermal_slowdown",
            getattr(nv, "nvmlClocksThrottleReasonSwThermalSlowdown", 0x20): "sw_thermal_slowdown",
            getattr(nv, "nvmlClocksThrottleReasonSwPowerCap", 0x4): "sw_power_cap",
            getattr(nv, "nvmlClocksThrottleReasonHwPowerBrakeSlowdown", 0x80): "hw_power_brake",
        }
        while not self.stop_flag.is_set():
            try:
                self.samples.append(float(nv.nvmlDeviceGetClockInfo(self.h, nv.NVML_CLOCK_SM)))
                r = int(nv.nvmlDeviceGetCurrentClocksThrottleReasons(self.h))
                for bit, name in names.items():
                    if r & bit:
                        self.reasons.add(name)
            except Exception:
                pass
            time.sleep(self.period)

    def finish(self):
        self.stop_flag.set()
        if self.is_alive():
            self.join()
        if not self.samples:
            return {"sm_mhz": None, "sm_max_mhz": self.max_mhz, "reasons": sorted(self.reasons), "samples": 0}
        s = sorted(self.samples)
        return {"sm_mhz": s[len(s) // 2], "sm_max_mhz": self.max_mhz, "reasons": sorted(self.reasons), "samples": len(s)}


# ------------------------------------------------------------------------------------------ our arm
def run_ours(args):
    import numpy as np
    import torch
    from paper_2411_18511_b200 import build, hr, inputs
    from paper_2411_18511_b200.dist import Ranks, whole_job_throughput
    from paper_2411_18511_b200.lattice import Lattice

    ranks = Ranks()
    assert ranks.world == args.gpus or ranks.world == 1, "launch N ranks with torchrun for --gpus N"
    dev_index = ranks.local_rank
    torch.cuda.set_device(dev_index)
    device = "cuda:%d" % dev_index
    build.build()
    hr.lib()

    L = (args.L,) * 4
    V = args.L ** 4
    Vh = V // 2
    kernel = {"auto": hr.KERNEL_AUTO, "generic": hr.KERNEL_GENERIC, "tiled": hr.KERNEL_TILED}[args.kernel]
    m0, m0c, csw = -0.2, -0.25, 1.2

    # ---- seeded synthetic inputs: configs[3] Haar links; configs[4] links exp(i 0.3 a.sigma)
    U = inputs.haar_gauge(L, 1)
    Uw = inputs.weak_gauge(L, 0.3, 1)
    psi = inputs.gaussian_spinor(L, 2, 2)

    S = {}
    for prec, tag in ((hr.PREC_F64, "f64"), (hr.PREC_F32, "f32")):
        lat = Lattice(L, hr.REP_FUND, prec, kernel, device)
        s = {"lat": lat, "U": lat.put_gauge_fund(U), "psi": lat.put_spinor(psi), "out": lat.empty_spinor(),
             "tmp": lat.empty_spinor(hr.ODD)}
        S[tag] = s
    lat64 = S["f64"]["lat"]
    S["f64"]["Uw"] = lat64.put_gauge_fund(Uw)
    S["f64"]["fwd"], S["f64"]["inv"] = lat64.clover_build(m0c, csw, S["f64"]["Uw"])
    S["f64"]["Uadj"] = lat64.empty_gauge(hr.REP_ADJ)
    torch.cuda.synchronize()
    del U, Uw
    st = hr.stream_ptr()

    # ---- the step: (name, precision, model op, output sites, callable)
    def mk(tag):
        s = S[tag]
        lat, g = s["lat"], s["lat"].g
        ev, od = lat.even, lat.odd
        ops = [
            ("hop_oe_" + tag, g, hr.OP_HOP, Vh, lambda: hr.hr_dirac_eo_apply(g, hr.EO_HOP_OE, 0.0, s["U"], None, None, ev(s["psi"]), od(s["out"]), None, st)),
            ("hop_eo_" + tag, g, hr.OP_HOP, Vh, lambda: hr.hr_dirac_eo_apply(g, hr.EO_HOP_EO, 0.0, s["U"], None, None, od(s["psi"]), ev(s["out"]), None, st)),
            ("dirac_" + tag, g, hr.OP_DIRAC, V, lambda: hr.hr_dirac_apply(g, m0, s["U"], s["psi"], s["out"], st)),
            ("dhat_" + tag, g, hr.OP_DHAT, Vh, lambda: hr.hr_dirac_eo_apply(g, hr.EO_DHAT, m0, s["U"], None, None, ev(s["psi"]), ev(s["out"]), s["tmp"], st)),
        ]
        if tag == "f64":
            ops += [
                ("clover_" + tag, g, hr.OP_CLOVER, V, lambda: hr.hr_clover_apply(g, hr.BOTH, s["fwd"], s["psi"], s["out"], st)),
                ("clover_inv_" + tag, g, hr.OP_CLOVER, V, lambda: hr.hr_clover_apply(g, hr.BOTH, s["inv"], s["psi"], s["out"], st)),
                ("dhat_clover_" + tag, g, hr.OP_DHAT_CLOVER, Vh, lambda: hr.hr_dirac_eo_apply(g, hr.EO_DHAT, m0c, s["Uw"], s["fwd"], s["inv"], ev(s["psi"]), ev(s["out"]), s["tmp"], st)),
                ("represent_" + tag, g, hr.OP_REPRESENT, V, lambda: hr.hr_represent_gauge(g, s["U"], s["Uadj"], st)),
            ]
        return ops

    ops = mk("f64") + mk("f32")
    model = {}
    for name, g, op, sites, _ in ops:
        f, bc, br = hr.hr_dirac_flops_bytes(g, op)
        model[name] = {"sites": sites, "flops": f * sites, "bytes": bc * sites, "bytes_requested": br * sites}
    step_bytes = sum(m["bytes"] for m in model.values())
    step_flops = sum(m["flops"] for m in model.values())
    step_sites = sum(m["sites"] for m in model.values())

    def step(events=None):
        for i, (name, g, op, sites, fn) in enumerate(ops):
            if events is not None:
                events[i][0].record()
            fn()
            if events is not None:
                events[i][1].record()

    for _ in range(max(3, args.warmup)):
        step()
    torch.cuda.synchronize()

    K = args.steps
    per_op_events = [[(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in ops] for _ in range(K)]
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    sampler = ClockSampler(dev_index)
    launches0 = hr.hr_launch_count()
    ranks.barrier()
    torch.cuda.synchronize()
    sampler.start()
    e0.record()
    for k in range(K):
        step(per_op_events[k])
    e1.record()
    torch.cuda.synchronize()
    ranks.barrier()
    clocks = sampler.finish()
    launches = hr.hr_launch_count() - launches0
    seconds = e0.elapsed_time(e1) * 1e-3
    value, tmax = whole_job_throughput(ranks, step_bytes * K / 1e9, seconds)
    ms_per_step = tmax * 1e3 / K

    op_report = {}
    for i, (name, g, op, sites, _) in enumerate(ops):
        ms = sum(per_op_events[k][i][0].elapsed_time(per_op_events[k][i][1]) for k in range(K)) / K
        m = model[name]
        op_report[name] = {
            "ms": round(ms, 4), "gbs": round(m["bytes"] / ms / 1e6, 1), "gbs_requested": round(m["bytes_requested"] / ms / 1e6, 1),
            "gflops": round(m["flops"] / ms / 1e6, 1), "gsites_per_s": round(m["sites"] / ms / 1e6, 3),
            "kernel": hr.hr_kernel_name(g) if "clover_" not in name[:7] and "represent" not in name else "site-diagonal",
        }

    # ---- roofline of the dominant kernel: the fp64 parity hop (2 launches per step as H1, same kernel inside E1/E2)
    peak, peak_src = peaks()
    hop_ms = 0.5 * (op_report["hop_oe_f64"]["ms"] + op_report["hop_eo_f64"]["ms"])
    hop_bytes = model["hop_oe_f64"]["bytes"]
    achieved = hop_bytes / hop_ms / 1e6
    traffic = None
    tp = os.path.join(ROOT, "profiles", "hop_f64_traffic.json")
    if os.path.exists(tp):
        try:
            with open(tp) as f:
                traffic = json.load(f).get(hr.hr_kernel_name(S["f64"]["lat"].g))
        except Exception:
            traffic = None
    roofline = {"bound": "hbm", "kernel": "parity hop fp64 (%s)" % hr.hr_kernel_name(S["f64"]["lat"].g), "achieved": round(achieved, 1),
                "peak": peak, "peak_source": peak_src, "unit": "GB/s", "frac": round(achieved / peak, 4),
                "frac_of_datasheet_8000": round(achieved / 8000.0, 4), "bytes_per_launch": hop_bytes,
                "avg_launch_ms": round(hop_ms, 4), "traffic": traffic,
                "fp32": {"achieved": round(model["hop_oe_f32"]["bytes"] / (0.5 * (op_report["hop_oe_f32"]["ms"] + op_report["hop_eo_f32"]["ms"])) / 1e6, 1)}}
    roofline["fp32"]["frac"] = round(roofline["fp32"]["achieved"] / peak, 4)
    # the same kernel timed as 30 back-to-back launches between ONE pair of events (no per-launch event gaps): context for
    # `achieved`, which is measured inside the step with an event pair around every launch
    b2b = {}
    for tag in ("f64", "f32"):
        fn = [o for o in ops if o[0] == "hop_oe_" + tag][0][4]
        for _ in range(3):
            fn()
        t0, t1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        t0.record()
        for _ in range(30):
            fn()
        t1.record()
        torch.cuda.synchronize()
        ms = t0.elapsed_time(t1) / 30
        b2b[tag] = {"avg_launch_ms": round(ms, 4), "achieved": round(model["hop_oe_" + tag]["bytes"] / ms / 1e6, 1),
                    "frac": round(model["hop_oe_" + tag]["bytes"] / ms / 1e6 / peak, 4)}
    roofline["back_to_back_30_launches"] = b2b

    # ---- end to end through the host-buffer C-ABI entry points (pinned host memory, copies inside the timed region)
    e2e = None
    if not args.no_e2e:
        e2e = run_e2e(args, ranks, hr, S, psi, L, m0, model)

    # ---- the parity configs, timed for the record (not part of the step): configs[1] 16^4 Dhat as a CUDA graph of
    # 100 repetitions (launch-bound: the lattice fits L2), configs[2] 24^4 adjoint with stored and on-the-fly links
    other = None
    if not args.no_other and ranks.rank == 0:
        try:
            other = other_configs(hr, inputs, Lattice)
            other.update(cg_report(hr, S, m0))
        except Exception as e:  # never let the side report break the bench line
            other = {"error": repr(e)}

    # ---- the oracle beside it (rank 0, N = 1 only)
    cpu = None
    if not args.no_cpu and ranks.rank == 0 and ranks.world == 1:
        cpu = cpu_baseline(L, m0, seconds_budget=15.0)

    if ranks.rank == 0:
        line = {
            "metric": METRIC, "value": round(value, 1), "unit": UNIT, "n_gpus": ranks.world, "steps": K, "warmup": max(3, args.warmup),
            "ms_per_step": round(ms_per_step, 4), "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
            "dtype": "f64+f32", "data": "synthetic",
            "config": {"workload": "configs[3]+[4]: %d^4 SU(2) fundamental, Haar links (clover: exp(i 0.3 a.sigma), csw 1.2); "
                                   "step = hop_oe, hop_eo, D, Dhat (f64 and f32) + clover, clover_inv, Dhat_clover, represent (f64)" % args.L,
                       "lattice": list(L), "l2_policy": "working set per op (>= 1.3 GB at 48^4) far exceeds the 126 MB L2; no flush needed",
                       "kernel": hr.hr_kernel_name(S["f64"]["lat"].g), "link_storage": "compressed first row (32 B fp64 / 16 B fp32)",
                       "parallelism": "replicas x%d (no data-path collective)" % ranks.world},
            "gflops": round(step_flops * K / tmax / 1e9 * ranks.world, 1),
            "gsites_per_s": round(step_sites * K / tmax / 1e9 * ranks.world, 3),
            "clocks": clocks, "gpu_launches": int(launches), "e2e": e2e, "roofline": roofline, "cpu_baseline": cpu, "ops": op_report, "other_configs": other,
        }
        print(json.dumps(line))
    ranks.close()


def other_configs(hr, inputs, Lattice):
    """per-apply device time of BASELINE.json configs[1] (16^4 fund, Dhat, 100 repetitions replayed as one CUDA graph)
    and configs[2] (24^4 adjoint: hop, D, Dhat; links stored as 3x3 reals and rebuilt on the fly)"""
    import torch
    out = {}
    reps = 100

    def timed(fn, n):
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        for _ in range(3):
            fn()
        torch.cuda.synchronize()
        e0.record()
        for _ in range(n):
            fn()
        e1.record()
        torch.cuda.synchronize()
        return e0.elapsed_time(e1) / n

    # configs[1]
    L = (16,) * 4
    U = inputs.weak_gauge(L, 0.3, 1)
    psi = inputs.gaussian_spinor(L, 2, 2)
    for prec, tag in ((hr.PREC_F64, "f64"), (hr.PREC_F32, "f32")):
        lat = Lattice(L, hr.REP_FUND, prec)
        g = lat.g
        U_dev, p_dev, o_dev, tmp = lat.put_gauge_fund(U), lat.put_spinor(psi), lat.empty_spinor(), lat.empty_spinor(hr.ODD)
        side = torch.cuda.Stream()
        side.wait_stream(torch.cuda.current_stream())
        with torch.cuda.stream(side):
            st = hr.stream_ptr(side)
            call = lambda: hr.hr_dirac_eo_apply(g, hr.EO_DHAT, -0.1, U_dev, None, None, lat.even(p_dev), lat.even(o_dev), tmp, st)
            call()
            side.synchronize()
            graph = torch.cuda.CUDAGraph()
            with torch.cuda.graph(graph, stream=side):
                stc = hr.stream_ptr(torch.cuda.current_stream())
                for _ in range(reps):
                    hr.hr_dirac_eo_apply(g, hr.EO_DHAT, -0.1, U_dev, None, None, lat.even(p_dev), lat.even(o_dev), tmp, stc)
        torch.cuda.current_stream().wait_stream(side)
        ms_graph = timed(graph.replay, 5) / reps
        st0 = hr.stream_ptr()
        ms_plain = timed(lambda: hr.hr_dirac_eo_apply(g, hr.EO_DHAT, -0.1, U_dev, None, None, lat.even(p_dev), lat.even(o_dev), tmp, st0), reps)
        f, bc, _ = hr.hr_dirac_flops_bytes(g, hr.OP_DHAT)
        sites = 16 ** 4 // 2
        out["config1_16^4_dhat_" + tag] = {"us_per_apply_graph": round(ms_graph * 1e3, 2), "us_per_apply_launches": round(ms_plain * 1e3, 2),
                                          "gsites_per_s": round(sites / ms_graph / 1e6, 3), "gflops": round(f * sites / ms_graph / 1e6, 1),
                                          "gbs_requested_from_l2": round(bc * sites / ms_graph / 1e6, 1), "kernel": hr.hr_kernel_name(g),
                                          "note": "fits L2 (24 MiB): HBM fraction not meaningful"}
    # configs[2]
    L = (24,) * 4
    V = 24 ** 4
    Uf = inputs.haar_gauge(L, 1)
    psi = inputs.gaussian_spinor(L, 3, 2)
    for storage, tag in ((hr.LINKS_COMPRESSED, "stored"), (hr.LINKS_ONTHEFLY, "onthefly")):
        lat = Lattice(L, hr.REP_ADJ, hr.PREC_F64, hr.KERNEL_AUTO, link_storage=storage)
        g = lat.g
        Uf_dev = lat.put_gauge_fund(Uf)
        U_dev = lat.represent(Uf_dev) if storage == hr.LINKS_COMPRESSED else Uf_dev
        p_dev, o_dev, tmp = lat.put_spinor(psi), lat.empty_spinor(), lat.empty_spinor(hr.ODD)
        st0 = hr.stream_ptr()
        for name, op, sites, fn in (
                ("hop", hr.OP_HOP, V // 2, lambda: hr.hr_dirac_eo_apply(g, hr.EO_HOP_OE, 0.0, U_dev, None, None, lat.even(p_dev), lat.odd(o_dev), None, st0)),
                ("dirac", hr.OP_DIRAC, V, lambda: hr.hr_dirac_apply(g, -0.3, U_dev, p_dev, o_dev, st0)),
                ("dhat", hr.OP_DHAT, V // 2, lambda: hr.hr_dirac_eo_apply(g, hr.EO_DHAT, -0.3, U_dev, None, None, lat.even(p_dev), lat.even(o_dev), tmp, st0))):
            ms = timed(fn, 50)
            f, bc, _ = hr.hr_dirac_flops_bytes(g, op)
            out["config2_24^4_adj_%s_%s_f64" % (name, tag)] = {"us_per_apply": round(ms * 1e3, 2), "gsites_per_s": round(sites / ms / 1e6, 3),
                                                            "gflops": round(f * sites / ms / 1e6, 1), "gbs": round(bc * sites / ms / 1e6, 1),
                                                            "kernel": hr.hr_kernel_name(g),
                                                            "note": "working set 0.1-0.2 GB: partly L2-resident, HBM fraction indicative only"}
    return out


def cg_report(hr, S, m0):
    """hr_cg_solve on the bench lattice: 20 iterations of CG on Dhat^dag Dhat, no convergence read-back
    in between; bytes per even site and iteration = 2 (5S + 16G) for the two Dhat + 11 S for the three vector kernels"""
    import torch
    out = {}
    for tag in ("f64", "f32"):
        s = S[tag]
        lat, g = s["lat"], s["lat"].g
        ws = hr.device_buffer(hr.hr_cg_workspace_bytes(g), lat.device)
        x = lat.empty_spinor(hr.EVEN)
        st = hr.stream_ptr()
        hr.hr_cg_solve(g, m0, s["U"], None, None, lat.even(s["psi"]), x, ws, 1e-30, 3, 1000, st)
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        n = 20
        e0.record()
        it, rel = hr.hr_cg_solve(g, m0, s["U"], None, None, lat.even(s["psi"]), x, ws, 1e-30, n, 1000, st)
        e1.record()
        torch.cuda.synchronize()
        ms = e0.elapsed_time(e1) / max(it, 1)
        _, bc, _ = hr.hr_dirac_flops_bytes(g, hr.OP_DHAT)
        w = 8 if tag == "f64" else 4
        bytes_site = 2 * bc + 11 * 16 * w
        Vh = lat.V // 2
        out["cg_48^4_" + tag] = {"ms_per_iteration": round(ms, 4), "iterations": it, "relres_after": rel,
                                 "gbs": round(bytes_site * Vh / ms / 1e6, 1), "bytes_per_even_site_per_iteration": bytes_site}
        del ws, x
    # H3c: the clover-improved full operator in one launch (not part of the step), fp64; bytes = H3 + clover blocks
    s64 = S["f64"]
    lat, g = s64["lat"], s64["lat"].g
    st = hr.stream_ptr()
    fn = lambda: hr.hr_dirac_clover_apply(g, s64["Uw"], s64["fwd"], s64["psi"], s64["out"], st)
    for _ in range(3):
        fn()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record()
    for _ in range(20):
        fn()
    e1.record()
    torch.cuda.synchronize()
    ms = e0.elapsed_time(e1) / 20
    _, bc, _ = hr.hr_dirac_flops_bytes(g, hr.OP_DIRAC)
    out["dirac_clover_48^4_f64"] = {"ms": round(ms, 4), "gbs": round((bc + 256.0) * lat.V / ms / 1e6, 1), "bytes_per_site": bc + 256.0}
    # time to a 1e-12 solution: plain fp64 CG against fp64 defect correction around fp32 CG (hr_cg_solve_mixed)
    s64, s32 = S["f64"], S["f32"]
    lat, g = s64["lat"], s64["lat"].g
    x = lat.empty_spinor(hr.EVEN)
    b = lat.even(s64["psi"])
    st = hr.stream_ptr()
    ws = hr.device_buffer(max(hr.hr_cg_workspace_bytes(g), hr.hr_cg_mixed_workspace_bytes(g)), lat.device)
    e0, e1, e2 = (torch.cuda.Event(enable_timing=True) for _ in range(3))
    e0.record()
    it, rel = hr.hr_cg_solve(g, m0, s64["U"], None, None, b, x, ws, 1e-12, 2000, 5, st)
    e1.record()
    no, ni, relm = hr.hr_cg_solve_mixed(g, m0, s64["U"], s32["U"], b, x, ws, 1e-12, 1e-4, 30, 2000, 5, st)
    e2.record()
    torch.cuda.synchronize()
    out["cg_48^4_to_1e-12"] = {"f64_ms": round(e0.elapsed_time(e1), 2), "f64_iterations": it, "f64_relres": rel,
                               "mixed_ms": round(e1.elapsed_time(e2), 2), "mixed_outer": no, "mixed_f32_iterations": ni,
                               "mixed_true_relres": relm}
    return out


def run_e2e(args, ranks, hr, S, psi, L, m0, model):
    """same metric through hr_dirac_apply_host / hr_dirac_eo_apply_host: canonical fields in pinned host memory,
    H2D + pack + operator + unpack + D2H inside the timed region, every step."""
    import numpy as np
    import torch
    from paper_2411_18511_b200 import inputs
    steps = max(1, min(args.steps, 3))
    total_s, total_bytes, h2d, d2h = 0.0, 0.0, 0, 0
    names = []
    U = inputs.haar_gauge(L, 1)
    for tag in ("f64", "f32"):
        lat = S[tag]["lat"]
        g = lat.g
        ws = hr.device_buffer(hr.hr_host_workspace_bytes(g), lat.device)
        Uh = torch.from_numpy(U.astype(lat.cplx)).pin_memory()
        ph = torch.from_numpy(psi.astype(lat.cplx)).pin_memory()
        oh = torch.empty_like(ph).pin_memory()
        st = hr.stream_ptr()
        calls = [("dirac_" + tag, lambda: hr.hr_dirac_apply_host(g, m0, Uh, ph, oh, ws, st)),
                 ("dhat_" + tag, lambda: hr.hr_dirac_eo_apply_host(g, hr.EO_DHAT, m0, Uh, ph, oh, ws, st))]
        for _, fn in calls:
            fn()  # warm-up (page-locks, first-touch)
        ranks.barrier()
        torch.cuda.synchronize()
        t0 = time.perf_counter()
        for _ in range(steps):
            for _, fn in calls:
                fn()  # each call synchronises its stream before returning
        torch.cuda.synchronize()
        total_s += time.perf_counter() - t0
        ranks.barrier()
        for name, _ in calls:
            total_bytes += model[name]["bytes"]
            names.append(name)
        h2d += len(calls) * (Uh.numel() * Uh.element_size() + ph.numel() * ph.element_size())
        d2h += len(calls) * (oh.numel() * oh.element_size())
        del ws, Uh, ph, oh
    from paper_2411_18511_b200.dist import whole_job_throughput
    value, tmax = whole_job_throughput(ranks, total_bytes * steps / 1e9, total_s)
    return {"value": round(value, 2), "unit": UNIT, "h2d_bytes_per_step": int(h2d), "d2h_bytes_per_step": int(d2h),
            "steps": steps, "ms_per_step": round(tmax * 1e3 / steps, 2), "ops": names,
            "note": "host canonical arrays -> H2D -> pack -> operator -> unpack -> D2H per call; bytes = same compulsory model"}


# ------------------------------------------------------------------------------------------ oracle timing
def oracle_sample(L, m0, nthreads, nsites):
    """time the oracle, as it stands, on a contiguous slab of `nsites` output sites of the 48^4 full-D workload"""
    import numpy as np
    import oracle
    from paper_2411_18511_b200 import inputs
    U = inputs.haar_gauge(L, 1)
    psi = inputs.gaussian_spinor(L, 2, 2)
    out = np.zeros_like(psi)
    oracle.lib()
    V = inputs.volume(L)
    nsites = min(nsites, V)
    oracle.dirac(L, 0, m0, U, psi, 0, min(4096, V), nthreads, out)  # touch
    return oracle, U, psi, out, nsites


def cpu_baseline(L, m0, seconds_budget=15.0):
    import oracle
    cores = oracle.available_cores()
    orc, U, psi, out, _ = oracle_sample(L, m0, cores, 0)
    V = 1
    for v in L:
        V *= v
    # calibrate on 1/64 of the lattice, then size the sample to the budget
    n0 = max(4096, V // 64)
    t = time.perf_counter()
    orc.dirac(L, 0, m0, U, psi, 0, n0, cores, out)
    dt = time.perf_counter() - t
    n = int(min(V, max(n0, n0 * seconds_budget * 0.5 / max(dt, 1e-6))))
    # about two thirds of the budget on all cores (repeated passes over the slab if one pass is short), the rest on one thread
    passes = max(1, int(seconds_budget * 0.66 / max(dt * n / n0, 1e-6)))
    t = time.perf_counter()
    for _ in range(passes):
        orc.dirac(L, 0, m0, U, psi, 0, n, cores, out)
    dt_all = (time.perf_counter() - t) / passes
    n1 = int(min(V, max(4096, n0 * seconds_budget * 0.33 / max(dt * cores, 1e-6))))
    t = time.perf_counter()
    orc.dirac(L, 0, m0, U, psi, 0, n1, 1, out)
    dt_one = time.perf_counter() - t
    bytes_per_site = 384.0  # same compulsory model as the GPU's fused full D, fp64, compressed links
    return {"value": round(n / dt_all * bytes_per_site / 1e9, 3), "unit": UNIT, "cores": cores, "kind": "oracle",
            "sample": "oracle full D (fp64) on the first %d of %d sites of the %d^4 workload, %d passes on %d threads (%.1f s) and %d sites on 1 thread (%.1f s); GB/s by the GPU's byte model (384 B/site)" % (n, V, L[0], passes, cores, dt_all * passes, n1, dt_one),
            "msites_per_s": round(n / dt_all / 1e6, 3), "single_thread_msites_per_s": round(n1 / dt_one / 1e6, 3),
            "label": "unoptimised CPU oracle, reported baseline, not a tuned CPU Dslash"}


def run_reference(args):
    """--impl reference: the oracle as it stands on the host cores; each step = full D on a bounded slab."""
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    import oracle
    L = (args.L,) * 4
    m0 = -0.2
    cores = oracle.available_cores()
    V = args.L ** 4
    orc, U, psi, out, _ = oracle_sample(L, m0, cores, 0)
    n0 = max(4096, V // 256)
    t = time.perf_counter()
    orc.dirac(L, 0, m0, U, psi, 0, n0, cores, out)
    dt = time.perf_counter() - t
    total_steps = args.steps + max(3, args.warmup)
    n = int(min(V, max(n0, n0 * (60.0 / total_steps) / max(dt, 1e-6))))   # whole run ~ 1 minute
    for _ in range(max(3, args.warmup)):
        orc.dirac(L, 0, m0, U, psi, 0, n, cores, out)
    t = time.perf_counter()
    for _ in range(args.steps):
        orc.dirac(L, 0, m0, U, psi, 0, n, cores, out)
    dt = time.perf_counter() - t
    value = n * args.steps / dt * 384.0 / 1e9
    sample = "oracle full D (fp64) on the first %d of %d sites of %d^4 per step, %d threads; GB/s by the 384 B/site compulsory model" % (n, V, args.L, cores)
    line = {
        "impl": "reference", "metric": METRIC, "value": round(value, 3), "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
        "warmup": max(3, args.warmup), "ms_per_step": round(dt * 1e3 / args.steps, 3), "higher_is_better": True, "scaling": "weak",
        "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": {"workload": "configs[3]: %d^4 SU(2) fundamental, Haar links; oracle (CPU) full D on a slab per step" % args.L,
                   "lattice": list(L), "parallelism": "host threads x%d" % cores},
        "cpu_baseline": {"value": round(value, 3), "unit": UNIT, "cores": cores, "kind": "oracle", "sample": sample},
        "e2e": {"value": round(value, 3), "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }
    print(json.dumps(line))


if __name__ == "__main__":
    a = parse()
    if a.impl == "reference":
        run_reference(a)
    else:
        run_ours(a)
