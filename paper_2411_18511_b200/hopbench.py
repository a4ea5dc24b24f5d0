"""Timing-only micro-benchmark of the hopping operators (the harness behind profiles/r01_tiled_variants.md).

    python -m paper_2411_18511_b200.hopbench [path/to/libhr_dslash.so]        (env HB_L: lattice extent, default 48)

Buffers of the right sizes filled with random numbers (the cost of the operators does not depend on the values);
per operator 5 warm-up launches, then 30 launches between one pair of CUDA events.  Prints microseconds per launch
of the bare parity hop, the full operator and the even-odd operator in fp64 and fp32, and the algorithmic GB/s.
To time a build variant: HR_NVCC_DEFS="-DHR_T_PIN_F64=1" python -m paper_2411_18511_b200.build --force, then this.
"""
from __future__ import annotations

import os
import sys

from . import hr


def bench(libpath=None, L=48, reps=30):
    import torch
    if libpath:
        hr._lib = None
        hr.LIB_PATH = os.path.abspath(libpath)
    hr.lib()
    out = {}
    for prec, tag in ((hr.PREC_F64, "f64"), (hr.PREC_F32, "f32")):
        g = hr.geom((L,) * 4, hr.REP_FUND, prec, hr.LINKS_COMPRESSED, hr.KERNEL_AUTO)
        U = torch.randn(hr.hr_gauge_bytes(g, hr.REP_FUND) // 4, device="cuda", dtype=torch.float32).view(torch.uint8)
        psi = torch.randn(hr.hr_spinor_bytes(g, hr.BOTH) // 4, device="cuda", dtype=torch.float32).view(torch.uint8)
        o = torch.empty_like(psi)
        half = psi.numel() // 2
        tmp = torch.empty(half, device="cuda", dtype=torch.uint8)
        st = hr.stream_ptr()
        ops = {"hop": lambda: hr.hr_dirac_eo_apply(g, hr.EO_HOP_OE, 0.0, U, None, None, psi[:half], o[half:], None, st),
               "dirac": lambda: hr.hr_dirac_apply(g, -0.2, U, psi, o, st),
               "dhat": lambda: hr.hr_dirac_eo_apply(g, hr.EO_DHAT, -0.2, U, None, None, psi[:half], o[:half], tmp, st)}
        for name, fn in ops.items():
            for _ in range(5):
                fn()
            torch.cuda.synchronize()
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            e0.record()
            for _ in range(reps):
                fn()
            e1.record()
            torch.cuda.synchronize()
            out[name + "_" + tag] = e0.elapsed_time(e1) / reps * 1e3
        out["kernel_" + tag] = hr.hr_kernel_name(g)
    return out


def main(argv):
    L = int(os.environ.get("HB_L", "48"))
    r = bench(argv[1] if len(argv) > 1 else None, L)
    V = L ** 4
    print(" ".join("%s %.1fus" % (k, v) for k, v in r.items() if not k.startswith("kernel")),
          "| hop f64 %.0f GB/s (%s), f32 %.0f GB/s (%s), D f64 %.0f GB/s" % (
              512 * V / 2 / r["hop_f64"] / 1e3, r["kernel_f64"], 256 * V / 2 / r["hop_f32"] / 1e3, r["kernel_f32"],
              384 * V / r["dirac_f64"] / 1e3))


if __name__ == "__main__":
    main(sys.argv)
