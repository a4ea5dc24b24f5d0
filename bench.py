#!/usr/bin/env python
"""bench.py — whole-hot-path benchmark of libhr_dslash on BASELINE.json configs[3]/[4] (48^4).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference] [--L 48]

One "step" = the fp64 Dslash group of BASELINE.json configs[3] over one 48^4 lattice of synthetic seeded fields (Haar
links, Gaussian spinors), inputs resident in HBM:  H1 hop o<-e, H1 hop e<-o, H3 full D, E1 Dhat  (5 kernel launches: Dhat is two hops).
`value` = compulsory (algorithmic) bytes of the step (hr_dirac_flops_bytes) / step time, in GB/s — the paper's
bandwidth metric; `dtype` = "f64".  The same four operators in fp32 and the clover / represent rows
(configs[4]: C2, C3, E2, H3c, R1) are timed right after, K steps each, and reported under `roofline.fp32_step`,
`roofline.clover_step` and per operator under `roofline.per_op` (fraction of the measured copy bandwidth and of the
8 TB/s datasheet figure, DRAM traffic from the ncu captures in profiles/kernel_traffic.json).
Prints ONE JSON line (rank 0).  See DESIGN.md §7 for every field.
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
IDLE_S = 1.0    # idle time that lets the board fall back below its power cap (burst state) before a side measurement


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
    ap.add_argument("--no-sustained", action="store_true", help="skip the 1.5 s sustained-load (power cap) timings")
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


def workload_config(L):
    """the `config` object, identical in both arms (the driver compares them)"""
    return {"workload": "BASELINE.json configs[3]: %d^4 periodic lattice, SU(2) fundamental, fp64, Haar-random links (seed 1), Gaussian spinor "
                        "(seed 2), m0 = -0.2; one step = hop o<-e, hop e<-o, full D, even-odd Dhat; GB/s by the compulsory byte model of "
                        "hr_dirac_flops_bytes (512 / 512 / 384 / 1152 B per output site, compressed links)" % L[0],
            "lattice": list(L), "ops": ["hop_oe", "hop_eo", "dirac", "dhat"], "precision": "fp64",
            "l2_policy": "working set per op (>= 1.3 GB at 48^4) far exceeds the 126 MB L2; no flush needed"}


GROUP_BYTES = {"hop_oe": 512.0, "hop_eo": 512.0, "dirac": 384.0, "dhat": 1152.0}   # fp64, per output site


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
    del Uw
    st = hr.stream_ptr()

    # ---- operator groups: (name, geometry, model op, output sites, extra bytes per site, callable)
    def dslash_group(tag):
        s = S[tag]
        lat, g = s["lat"], s["lat"].g
        ev, od = lat.even, lat.odd
        return [
            ("hop_oe_" + tag, g, hr.OP_HOP, Vh, 0.0, lambda: hr.hr_dirac_eo_apply(g, hr.EO_HOP_OE, 0.0, s["U"], None, None, ev(s["psi"]), od(s["out"]), None, st)),
            ("hop_eo_" + tag, g, hr.OP_HOP, Vh, 0.0, lambda: hr.hr_dirac_eo_apply(g, hr.EO_HOP_EO, 0.0, s["U"], None, None, od(s["psi"]), ev(s["out"]), None, st)),
            ("dirac_" + tag, g, hr.OP_DIRAC, V, 0.0, lambda: hr.hr_dirac_apply(g, m0, s["U"], s["psi"], s["out"], st)),
            ("dhat_" + tag, g, hr.OP_DHAT, Vh, 0.0, lambda: hr.hr_dirac_eo_apply(g, hr.EO_DHAT, m0, s["U"], None, None, ev(s["psi"]), ev(s["out"]), s["tmp"], st)),
        ]

    def clover_group():
        s = S["f64"]
        lat, g = s["lat"], s["lat"].g
        ev = lat.even
        blk = hr.hr_dirac_flops_bytes(g, hr.OP_CLOVER)[1] - 2 * 128.0        # block bytes per site
        return [
            ("clover_f64", g, hr.OP_CLOVER, V, 0.0, lambda: hr.hr_clover_apply(g, hr.BOTH, s["fwd"], s["psi"], s["out"], st)),
            ("clover_inv_f64", g, hr.OP_CLOVER, V, 0.0, lambda: hr.hr_clover_apply(g, hr.BOTH, s["inv"], s["psi"], s["out"], st)),
            ("dhat_clover_f64", g, hr.OP_DHAT_CLOVER, Vh, 0.0, lambda: hr.hr_dirac_eo_apply(g, hr.EO_DHAT, m0c, s["Uw"], s["fwd"], s["inv"], ev(s["psi"]), ev(s["out"]), s["tmp"], st)),
            ("dirac_clover_f64", g, hr.OP_DIRAC, V, blk, lambda: hr.hr_dirac_clover_apply(g, s["Uw"], s["fwd"], s["psi"], s["out"], st)),
            ("represent_f64", g, hr.OP_REPRESENT, V, 0.0, lambda: hr.hr_represent_gauge(g, s["U"], s["Uadj"], st)),
        ]

    groups = {"f64": dslash_group("f64"), "f32": dslash_group("f32"), "clover": clover_group()}
    model = {}
    for ops in groups.values():
        for name, g, op, sites, extra, _ in ops:
            f, bc, br = hr.hr_dirac_flops_bytes(g, op)
            if name == "dirac_clover_f64":
                f += hr.hr_dirac_flops_bytes(g, hr.OP_CLOVER)[0] - 3 * 16.0      # A psi replaces the (4+m0) psi axpy
            model[name] = {"sites": sites, "flops": f * sites, "bytes": (bc + extra) * sites, "bytes_requested": (br + extra) * sites}

    def totals(ops):
        return tuple(sum(model[o[0]][k] for o in ops) for k in ("bytes", "flops", "sites"))

    def step(ops, events=None):
        for i, o in enumerate(ops):
            if events is not None:
                events[i][0].record()
            o[5]()
            if events is not None:
                events[i][1].record()

    def timed_group(ops, K, count_launches=False):
        """K steps of one group between a barrier + synchronize on both sides; per-launch event pairs inside"""
        evs = [[(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in ops] for _ in range(K)]
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        sampler = ClockSampler(dev_index) if count_launches else None
        n0 = hr.hr_launch_count()
        ranks.barrier()
        torch.cuda.synchronize()
        if sampler:
            sampler.start()
        e0.record()
        for k in range(K):
            step(ops, evs[k])
        e1.record()
        torch.cuda.synchronize()
        ranks.barrier()
        clocks = sampler.finish() if sampler else None
        launches = hr.hr_launch_count() - n0
        per_op = [sum(evs[k][i][0].elapsed_time(evs[k][i][1]) for k in range(K)) / K for i in range(len(ops))]
        return e0.elapsed_time(e1) * 1e-3, per_op, launches, clocks

    W, K = max(3, args.warmup), args.steps
    for _ in range(W):
        for ops in groups.values():
            step(ops)
    for _ in range(W):       # the headline group is warmed up last, so the timed region starts from its own steady state
        step(groups["f64"])
    torch.cuda.synchronize()

    seconds, ms64, launches, clocks = timed_group(groups["f64"], K, count_launches=True)
    step_bytes, step_flops, step_sites = totals(groups["f64"])
    value, tmax = whole_job_throughput(ranks, step_bytes * K / 1e9, seconds)
    ms_per_step = tmax * 1e3 / K
    side = {}
    op_ms = dict(zip([o[0] for o in groups["f64"]], ms64))
    # Side groups are timed the way the headline group is: from an idle power state (IDLE_S seconds without work), after W warm-up
    # steps of their own.  Without the pause they would start inside the board's 1000 W power cap, which the warm-up and the
    # headline group have reached by then (SM clock 1965 -> 1400-1600 MHz after ~0.4 s of these kernels: `sustained_under_power_cap`).
    for key in ("f32", "clover"):
        torch.cuda.synchronize()
        time.sleep(IDLE_S)
        for _ in range(W):
            step(groups[key])
        sec, ms, _, ck = timed_group(groups[key], K, count_launches=True)
        by, fl, si = totals(groups[key])
        side[key] = {"value": round(by * K / sec / 1e9, 1), "unit": UNIT, "ms_per_step": round(sec * 1e3 / K, 4),
                     "gflops": round(fl * K / sec / 1e9, 1), "gsites_per_s": round(si * K / sec / 1e9, 3), "ops": [o[0] for o in groups[key]],
                     "clocks": ck, "idle_before_s": IDLE_S}
        op_ms.update(zip([o[0] for o in groups[key]], ms))

    # ---- per-operator report and roofline (HBM-bound: DESIGN.md §5); DRAM traffic per launch from the committed ncu captures
    peak, peak_src = peaks()
    traffic_db = {}
    tp = os.path.join(ROOT, "profiles", "kernel_traffic.json")
    if os.path.exists(tp):
        try:
            with open(tp) as f:
                traffic_db = json.load(f)
        except Exception:
            traffic_db = {}
    kname = hr.hr_kernel_name(S["f64"]["lat"].g)
    per_op = {}
    for name, ms in op_ms.items():
        m = model[name]
        gbs = m["bytes"] / ms / 1e6
        tr = traffic_db.get(kname, {}).get(name) if args.L == 48 else None
        per_op[name] = {"ms": round(ms, 4), "gbs": round(gbs, 1), "frac": round(gbs / peak, 4), "frac_of_8000": round(gbs / 8000.0, 4),
                        "gflops": round(m["flops"] / ms / 1e6, 1), "gsites_per_s": round(m["sites"] / ms / 1e6, 3),
                        "bytes_per_launch_set": m["bytes"], "traffic": tr, "traffic_ratio": round(tr / m["bytes"], 4) if tr else None}
    hop_ms = 0.5 * (op_ms["hop_oe_f64"] + op_ms["hop_eo_f64"])
    hop_bytes = model["hop_oe_f64"]["bytes"]
    achieved = hop_bytes / hop_ms / 1e6
    roofline = {"bound": "hbm", "kernel": "parity hop fp64 (%s): 4 of the 5 launches of the step and %d%% of its time" % (
                    kname, round(100 * (op_ms["hop_oe_f64"] + op_ms["hop_eo_f64"] + op_ms["dhat_f64"]) / sum(ms64))),
                "achieved": round(achieved, 1), "peak": peak, "peak_source": peak_src, "unit": "GB/s", "frac": round(achieved / peak, 4),
                "frac_of_datasheet_8000": round(achieved / 8000.0, 4), "bytes_per_launch": hop_bytes, "avg_launch_ms": round(hop_ms, 4),
                "traffic": per_op["hop_oe_f64"]["traffic"], "per_op": per_op, "fp32_step": side["f32"], "clover_step": side["clover"]}
    # the hop kernels timed as 30 back-to-back launches between ONE pair of events (no per-launch event gaps), each parity on
    # its own: context for `achieved`, and the check that o<-e and e<-o cost the same when neither follows another operator
    b2b = {}
    for name in ("hop_oe_f64", "hop_eo_f64", "dirac_f64", "hop_oe_f32", "hop_eo_f32", "dirac_f32"):
        fn = [o for ops in groups.values() for o in ops if o[0] == name][0][5]
        torch.cuda.synchronize()
        time.sleep(0.25)      # burst regime: every operator starts below the power cap
        for _ in range(3):
            fn()
        t0, t1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        t0.record()
        for _ in range(30):
            fn()
        t1.record()
        torch.cuda.synchronize()
        ms = t0.elapsed_time(t1) / 30
        b2b[name] = {"avg_launch_ms": round(ms, 4), "gbs": round(model[name]["bytes"] / ms / 1e6, 1), "frac": round(model[name]["bytes"] / ms / 1e6 / peak, 4)}
    roofline["back_to_back_30_launches"] = b2b
    # the same launches under sustained load: ~1.5 s of one operator back to back; the board reaches its power limit, NVML reports
    # sw_power_cap and the SM clock drops while the memory clock stays
    sustained = {}
    if not args.no_sustained:
        for name in ("hop_oe_f64", "dirac_f64", "dirac_f32"):
            fn = [o for ops in groups.values() for o in ops if o[0] == name][0][5]
            torch.cuda.synchronize()
            time.sleep(IDLE_S)
            t_end = time.time() + 1.5
            while time.time() < t_end:
                for _ in range(100):
                    fn()
                torch.cuda.synchronize()
            sampler = ClockSampler(dev_index)
            sampler.start()
            t0, t1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            t0.record()
            for _ in range(300):
                fn()
            t1.record()
            torch.cuda.synchronize()
            ck = sampler.finish()
            ms = t0.elapsed_time(t1) / 300
            sustained[name] = {"avg_launch_ms": round(ms, 4), "gbs": round(model[name]["bytes"] / ms / 1e6, 1), "sm_mhz": ck["sm_mhz"],
                               "reasons": ck["reasons"]}
    roofline["sustained_under_power_cap"] = sustained

    # ---- end to end through the host-buffer C-ABI entry points (pinned host memory, copies inside the timed region)
    e2e = None
    if not args.no_e2e:
        e2e = run_e2e(args, ranks, hr, S, U, psi, L, m0, model)
    del U

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
        cfg = workload_config(L)
        line = {
            "metric": METRIC, "value": round(value, 1), "unit": UNIT, "n_gpus": ranks.world, "steps": K, "warmup": W,
            "ms_per_step": round(ms_per_step, 4), "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
            "dtype": "f64", "data": "synthetic", "config": cfg,
            "impl_detail": {"kernel": kname, "link_storage": "compressed first row (32 B fp64 / 16 B fp32)",
                            "parallelism": "replicas x%d (no data-path collective)" % ranks.world,
                            "plan_hop": hr.hr_kernel_plan(S["f64"]["lat"].g, hr.OP_HOP), "plan_dirac": hr.hr_kernel_plan(S["f64"]["lat"].g, hr.OP_DIRAC)},
            "gflops": round(step_flops * K / tmax / 1e9 * ranks.world, 1),
            "gsites_per_s": round(step_sites * K / tmax / 1e9 * ranks.world, 3),
            "clocks": clocks, "gpu_launches": int(launches), "e2e": e2e, "roofline": roofline, "cpu_baseline": cpu,
            "fp32": side["f32"], "clover": side["clover"], "other_configs": other,
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
        torch.cuda.synchronize()
        time.sleep(0.25)          # every side row starts below the power cap (burst regime, as the back-to-back table)
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
    # 48^4 adjoint fermions (the paper's local volume; higher representations are HiRep's purpose):
    # HBM-sized, so the fraction of the measured copy bandwidth is meaningful here
    import json as _json
    peak = peaks()[0]
    L = (48,) * 4
    V = 48 ** 4
    for prec, ptag in ((hr.PREC_F64, "f64"), (hr.PREC_F32, "f32")):
        for storage, tag in ((hr.LINKS_COMPRESSED, "stored"), (hr.LINKS_ONTHEFLY, "onthefly")):
            lat = Lattice(L, hr.REP_ADJ, prec, hr.KERNEL_AUTO, link_storage=storage)
            g = lat.g
            # timing only: random bytes of the right sizes (the cost is value-independent; parity is tests/test_gpu_parity.py)
            Uf_dev = torch.randn(hr.hr_gauge_bytes(g, hr.REP_FUND) // 4, device="cuda").view(torch.uint8)
            U_dev = lat.represent(Uf_dev) if storage == hr.LINKS_COMPRESSED else Uf_dev
            p_dev = torch.randn(hr.hr_spinor_bytes(g, hr.BOTH) // 4, device="cuda").view(torch.uint8)
            o_dev, tmp = lat.empty_spinor(), lat.empty_spinor(hr.ODD)
            st0 = hr.stream_ptr()
            for name, op, sites, fn in (
                    ("hop", hr.OP_HOP, V // 2, lambda: hr.hr_dirac_eo_apply(g, hr.EO_HOP_OE, 0.0, U_dev, None, None, lat.even(p_dev), lat.odd(o_dev), None, st0)),
                    ("dirac", hr.OP_DIRAC, V, lambda: hr.hr_dirac_apply(g, -0.3, U_dev, p_dev, o_dev, st0)),
                    ("dhat", hr.OP_DHAT, V // 2, lambda: hr.hr_dirac_eo_apply(g, hr.EO_DHAT, -0.3, U_dev, None, None, lat.even(p_dev), lat.even(o_dev), tmp, st0))):
                ms = timed(fn, 20)
                f, bc, _ = hr.hr_dirac_flops_bytes(g, op)
                out["adjoint_48^4_%s_%s_%s" % (name, tag, ptag)] = {"us_per_apply": round(ms * 1e3, 1), "gsites_per_s": round(sites / ms / 1e6, 3),
                                                                    "gflops": round(f * sites / ms / 1e6, 1), "gbs": round(bc * sites / ms / 1e6, 1),
                                                                    "frac": round(bc * sites / ms / 1e6 / peak, 4), "bytes_per_site": bc,
                                                                    "kernel": hr.hr_kernel_name(g)}
            del Uf_dev, U_dev, p_dev, o_dev, tmp
    # complex 3 x 3 links (HR_REP_SU3, DESIGN.md §1 row f4b) at the same volume: generic kernel, links stored in full or as two rows
    for prec, storage, ptag in ((hr.PREC_F64, hr.LINKS_FULL, "f64"), (hr.PREC_F32, hr.LINKS_FULL, "f32"),
                                (hr.PREC_F64, hr.LINKS_COMPRESSED, "tworows_f64"), (hr.PREC_F32, hr.LINKS_COMPRESSED, "tworows_f32")):
        lat = Lattice(L, hr.REP_SU3, prec, hr.KERNEL_AUTO, link_storage=storage)
        g = lat.g
        U_dev = torch.randn(hr.hr_gauge_bytes(g, hr.REP_SU3) // 4, device="cuda").view(torch.uint8)
        p_dev = torch.randn(hr.hr_spinor_bytes(g, hr.BOTH) // 4, device="cuda").view(torch.uint8)
        o_dev, tmp = lat.empty_spinor(), lat.empty_spinor(hr.ODD)
        st0 = hr.stream_ptr()
        for name, op, sites, fn in (
                ("hop", hr.OP_HOP, V // 2, lambda: hr.hr_dirac_eo_apply(g, hr.EO_HOP_OE, 0.0, U_dev, None, None, lat.even(p_dev), lat.odd(o_dev), None, st0)),
                ("dirac", hr.OP_DIRAC, V, lambda: hr.hr_dirac_apply(g, -0.3, U_dev, p_dev, o_dev, st0)),
                ("dhat", hr.OP_DHAT, V // 2, lambda: hr.hr_dirac_eo_apply(g, hr.EO_DHAT, -0.3, U_dev, None, None, lat.even(p_dev), lat.even(o_dev), tmp, st0))):
            ms = timed(fn, 20)
            f, bc, _ = hr.hr_dirac_flops_bytes(g, op)
            out["su3_48^4_%s_%s" % (name, ptag)] = {"us_per_apply": round(ms * 1e3, 1), "gsites_per_s": round(sites / ms / 1e6, 3),
                                                   "gflops": round(f * sites / ms / 1e6, 1), "gbs": round(bc * sites / ms / 1e6, 1),
                                                   "frac": round(bc * sites / ms / 1e6 / peak, 4), "bytes_per_site": bc, "kernel": hr.hr_kernel_name(g)}
        # the two-index antisymmetric representation of the links (hr_represent_gauge_antisym): a streaming kernel that reads and
        # writes one gauge field — bytes per link = 2 x the stored link
        R_dev = lat.empty_gauge(hr.REP_SU3)
        ms = timed(lambda: hr.hr_represent_gauge_antisym(g, U_dev, R_dev, st0), 20)
        rbytes = 2.0 * hr.hr_gauge_bytes(g, hr.REP_SU3)
        out["su3_48^4_represent_antisym_%s" % ptag] = {"us_per_apply": round(ms * 1e3, 1), "gbs": round(rbytes / ms / 1e6, 1),
                                                       "frac": round(rbytes / ms / 1e6 / peak, 4), "bytes_per_link": rbytes / (4 * V)}
        del U_dev, p_dev, o_dev, tmp, R_dev
    # the sharded hop on this one GPU: a 48^4 local lattice whose four directions are all cut onto the rank itself;
    # pack + device-to-device face copies + interior kernel + boundary kernels per hop o<-e, in order and with pack / copies
    # on a side stream (no multi-GPU hardware in this run: this measures what a cut costs a rank, not the transport)
    from paper_2411_18511_b200 import halo
    for prec, ptag in ((hr.PREC_F64, "f64"), (hr.PREC_F32, "f32")):
        lat = Lattice(L, hr.REP_FUND, prec, hr.KERNEL_AUTO)
        g = lat.g
        U_dev = torch.randn(hr.hr_gauge_bytes(g, hr.REP_FUND) // 4, device="cuda").view(torch.uint8)
        p_dev = torch.randn(hr.hr_spinor_bytes(g, hr.BOTH) // 4, device="cuda").view(torch.uint8)
        o_dev = lat.empty_spinor()
        for split in ((1, 0, 0, 0), (1, 1, 1, 0), (1, 1, 1, 1)):
            sh = halo.Shard(lat, (1, 1, 1, 1), (0, 0, 0, 0), split)
            shards, Ud, ind, outd = {(0, 0, 0, 0): sh}, {(0, 0, 0, 0): U_dev}, {(0, 0, 0, 0): lat.even(p_dev)}, {(0, 0, 0, 0): lat.odd(o_dev)}
            ms_seq = timed(lambda: halo.hop_all(shards, halo.exchange_in_process, hr.ODD, Ud, ind, outd), 20)
            ms_ovl = timed(lambda: halo.hop_all(shards, halo.exchange_in_process, hr.ODD, Ud, ind, outd, overlap=True), 20)
            out["sharded_hop_48^4_local_%dcuts_%s" % (sum(split), ptag)] = {
                "us_in_order": round(ms_seq * 1e3, 1), "us_overlapped": round(ms_ovl * 1e3, 1),
                "face_bytes": hr.hr_halo_face_bytes(g, 0), "faces_per_hop": 2 * sum(split), "interior_kernel": hr.hr_kernel_name(g)}
        del U_dev, p_dev, o_dev
    return out


def cg_report(hr, S, m0):
    """hr_cg_solve on the bench lattice: 20 iterations of CG on Dhat^dag Dhat, no convergence read-back
    in between; bytes per even site and iteration = 2 (5S + 16G) for the four hops of the two Dhat + 6 S: the CG update riding in the
    last hop's epilogue reads and writes r instead of writing Dhat s (1 S net), and x += alpha p, p = r + beta p share the one vector kernel (5 S)"""
    import torch
    out = {}
    for tag in ("f64", "f32"):
        s = S[tag]
        lat, g = s["lat"], s["lat"].g
        ws = hr.device_buffer(hr.hr_cg_workspace_bytes(g), lat.device)
        x = lat.empty_spinor(hr.EVEN)
        st = hr.stream_ptr()
        torch.cuda.synchronize()
        time.sleep(0.5)          # burst regime, as every side row
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
        bytes_site = 2 * bc + 6 * 16 * w
        Vh = lat.V // 2
        out["cg_48^4_" + tag] = {"ms_per_iteration": round(ms, 4), "iterations": it, "relres_after": rel,
                                 "gbs": round(bytes_site * Vh / ms / 1e6, 1), "bytes_per_even_site_per_iteration": bytes_site}
        del ws, x
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


def run_e2e(args, ranks, hr, S, U, psi, L, m0, model):
    """the headline metric end to end through the host-buffer C-ABI: canonical fp64 fields in pinned host memory; every
    step uploads its inputs and downloads its results inside the timed region.  Two readings:
      gauge resident (the headline e2e value): hr_gauge_upload_host once (untimed: the gauge field changes once per
        molecular-dynamics step), then per step ONE hr_apply_host_ops call over NRHS right-hand sides for each of the
        step's operators (hop o<-e, hop e<-o, D, Dhat: 16 items) — H2D, pack, operator, unpack, D2H pipelined over three streams;
      gauge included: hr_dirac_apply_host + hr_dirac_eo_apply_host, which also upload the links on every call."""
    import torch
    from paper_2411_18511_b200.dist import whole_job_throughput
    steps = max(1, min(args.steps, 3))
    nrhs = 4
    lat = S["f64"]["lat"]
    g, st = lat.g, hr.stream_ptr()
    Uh = torch.from_numpy(U.astype(lat.cplx)).pin_memory()
    ins = [torch.from_numpy(psi.astype(lat.cplx)).pin_memory()]
    for i in range(1, nrhs):
        ins.append(torch.roll(ins[0], i, 0).contiguous().pin_memory())
    outs = [torch.empty_like(a).pin_memory() for a in ins]
    nbytes = ins[0].numel() * ins[0].element_size()
    # ---- gauge resident
    u_dev = lat.empty_gauge(hr.REP_FUND)
    ws = hr.device_buffer(max(hr.hr_host_batch_workspace_bytes(g), hr.hr_canonical_gauge_bytes(g, hr.REP_FUND)), lat.device)
    hr.hr_gauge_upload_host(g, hr.REP_FUND, Uh, u_dev, ws, st)
    calls = [("hop_oe_f64", hr.EO_HOP_OE), ("hop_eo_f64", hr.EO_HOP_EO), ("dirac_f64", hr.HOST_DIRAC), ("dhat_f64", hr.EO_DHAT)]

    step_ops = [op for _, op in calls for _ in range(nrhs)]
    step_ins, step_outs = ins * len(calls), outs * len(calls)

    def resident_step():      # ONE pipeline over the 16 items of the step (hr_apply_host_ops): fill and drain are paid once
        hr.hr_apply_host_ops(g, step_ops, m0, u_dev, None, None, step_ins, step_outs, ws, st)

    resident_step()   # warm-up (page-locks, first-touch, stream creation)
    ranks.barrier()
    torch.cuda.synchronize()
    t0 = time.perf_counter()
    for _ in range(steps):
        resident_step()
    torch.cuda.synchronize()
    sec = time.perf_counter() - t0
    ranks.barrier()
    by = sum(model[name]["bytes"] for name, _ in calls) * nrhs
    value, tmax = whole_job_throughput(ranks, by * steps / 1e9, sec)
    h2d = d2h = len(calls) * nrhs * nbytes
    del u_dev, ws
    # ---- gauge included (the round-1 path), one right-hand side per call
    ws = hr.device_buffer(hr.hr_host_workspace_bytes(g), lat.device)
    old = [("dirac_f64", lambda: hr.hr_dirac_apply_host(g, m0, Uh, ins[0], outs[0], ws, st)),
           ("dhat_f64", lambda: hr.hr_dirac_eo_apply_host(g, hr.EO_DHAT, m0, Uh, ins[0], outs[0], ws, st))]
    for _, fn in old:
        fn()
    torch.cuda.synchronize()
    t0 = time.perf_counter()
    for _, fn in old:
        fn()
    torch.cuda.synchronize()
    sec_old = time.perf_counter() - t0
    by_old = sum(model[name]["bytes"] for name, _ in old)
    gauge_bytes = Uh.numel() * Uh.element_size()
    del ws
    return {"value": round(value, 2), "unit": UNIT, "h2d_bytes_per_step": int(h2d), "d2h_bytes_per_step": int(d2h),
            "steps": steps, "ms_per_step": round(tmax * 1e3 / steps, 2), "ops": [n for n, _ in calls], "nrhs_per_op": nrhs,
            "pcie_gbs_each_direction": round(h2d * steps / tmax / 1e9, 1),
            "gauge_included": {"value": round(by_old / sec_old / 1e9, 2), "unit": UNIT, "ops": [n for n, _ in old],
                               "h2d_bytes": int(len(old) * (gauge_bytes + nbytes)), "d2h_bytes": int(len(old) * nbytes), "ms": round(sec_old * 1e3, 2)},
            "note": "gauge resident on the device (uploaded once per gauge update), the 16 items of the step (4 right-hand sides per operator) in ONE "
                    "hr_apply_host_ops pipeline H2D | pack+operator+unpack | D2H; GB/s by the same compulsory byte model as `value`; PCIe-bound by construction"}


# ------------------------------------------------------------------------------------------ oracle timing
class OracleStep:
    """the headline step (hop o<-e, hop e<-o, full D, Dhat; fp64) on the oracle as it stands, on the first `nplanes` x0-planes
    of the lattice (all of it when nplanes == L0).  On a slab, Dhat is composed from the oracle's own hop: H_oe on the slab and
    its two neighbour planes, H_eo on the slab, then (4+m0) psi_e - H_eo H_oe psi_e / (4 (4+m0))."""

    def __init__(self, L, m0):
        import numpy as np
        import oracle
        from paper_2411_18511_b200 import inputs
        self.np, self.orc, self.L, self.m0 = np, oracle, L, m0
        self.V = inputs.volume(L)
        self.s0 = self.V // L[0]
        self.U = inputs.haar_gauge(L, 1)
        self.psi = inputs.gaussian_spinor(L, 2, 2)
        self.even = (inputs.site_parity(L) == 0)[:, None, None]
        self.psi_e = np.where(self.even, self.psi, 0.0)
        self.out = np.zeros_like(self.psi)
        self.t = np.zeros_like(self.psi)
        oracle.lib()
        self.cores = oracle.available_cores()
        oracle.dirac(L, 0, m0, self.U, self.psi, 0, min(4096, self.V), self.cores, self.out)  # touch

    def bytes(self, nplanes):
        n = nplanes * self.s0
        return n / 2 * (GROUP_BYTES["hop_oe"] + GROUP_BYTES["hop_eo"] + GROUP_BYTES["dhat"]) + n * GROUP_BYTES["dirac"]

    def run(self, nplanes, threads):
        o, L, m0, d = self.orc, self.L, self.m0, 4.0 + self.m0
        n = nplanes * self.s0
        o.hop(L, 0, 1, self.U, self.psi, 0, n, threads, self.out)
        o.hop(L, 0, 0, self.U, self.psi, 0, n, threads, self.out)
        o.dirac(L, 0, m0, self.U, self.psi, 0, n, threads, self.out)
        if nplanes == L[0]:
            o.dirac_eo(L, 0, m0, self.U, self.psi, threads)
        else:
            o.hop(L, 0, 1, self.U, self.psi_e, 0, min(self.V, n + self.s0), threads, self.t)
            o.hop(L, 0, 1, self.U, self.psi_e, self.V - self.s0, self.V, threads, self.t)
            o.hop(L, 0, 0, self.U, self.t, 0, n, threads, self.out)
            self.out[:n] = self.np.where(self.even[:n], d * self.psi_e[:n] - self.out[:n] / (4.0 * d), 0.0)

    def planes_for(self, seconds, threads):
        """how many x0-planes one step may cover to take about `seconds` (calibrated on one plane)"""
        t = time.perf_counter()
        self.run(1, threads)
        dt = max(time.perf_counter() - t, 1e-6)
        return int(max(1, min(self.L[0], seconds / dt)))


def cpu_baseline(L, m0, seconds_budget=15.0):
    w = OracleStep(L, m0)
    cores = w.cores
    npl = w.planes_for(seconds_budget * 0.6 / 2, cores)        # two passes on all cores
    passes = 2
    t = time.perf_counter()
    for _ in range(passes):
        w.run(npl, cores)
    dt_all = (time.perf_counter() - t) / passes
    npl1 = w.planes_for(seconds_budget * 0.3, 1)
    t = time.perf_counter()
    w.run(npl1, 1)
    dt_one = time.perf_counter() - t
    return {"value": round(w.bytes(npl) / dt_all / 1e9, 3), "unit": UNIT, "cores": cores, "kind": "oracle",
            "sample": "the step's four operators (hop o<-e, hop e<-o, D, Dhat; fp64) by the oracle on the first %d of %d x0-planes of the %d^4 "
                      "workload, %d passes on %d threads (%.1f s per pass), and on %d plane(s) on 1 thread (%.1f s); GB/s by the same byte "
                      "model as `value`" % (npl, L[0], L[0], passes, cores, dt_all, npl1, dt_one),
            "single_thread_value": round(w.bytes(npl1) / dt_one / 1e9, 3),
            "label": "unoptimised CPU oracle, reported baseline, not a tuned CPU Dslash"}


def run_reference(args):
    """--impl reference: the oracle as it stands on the host cores, same step (hop o<-e, hop e<-o, D, Dhat; fp64), same config,
    metric and unit as our arm; each step covers a bounded number of x0-planes so that the run ends within a few minutes."""
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    L = (args.L,) * 4
    m0 = -0.2
    w = OracleStep(L, m0)
    W = max(3, args.warmup)
    npl = w.planes_for(90.0 / (args.steps + W), w.cores)     # whole run ~ 1.5 minutes at most
    for _ in range(W):
        w.run(npl, w.cores)
    t = time.perf_counter()
    for _ in range(args.steps):
        w.run(npl, w.cores)
    dt = time.perf_counter() - t
    value = w.bytes(npl) * args.steps / dt / 1e9
    sample = "the step's four operators by the oracle on the first %d of %d x0-planes of %d^4 per step, %d threads; GB/s by the same byte model" % (
        npl, L[0], args.L, w.cores)
    line = {
        "impl": "reference", "metric": METRIC, "value": round(value, 3), "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
        "warmup": W, "ms_per_step": round(dt * 1e3 / args.steps, 3), "higher_is_better": True, "scaling": "weak",
        "vs_baseline": None, "dtype": "f64", "data": "synthetic", "config": workload_config(L),
        "impl_detail": {"parallelism": "host threads x%d" % w.cores, "planes_per_step": npl},
        "cpu_baseline": {"value": round(value, 3), "unit": UNIT, "cores": w.cores, "kind": "oracle", "sample": sample},
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
