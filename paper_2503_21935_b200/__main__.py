"""Standalone application (Fig. 1 diagram 1: random numbers, phase-space sampling and the ME
calculation all data parallel): seeded RAMBO points made on the device by me_generate, the matrix elements by
me_compute, nothing on the host.

    python -m paper_2503_21935_b200 --process gg_ttgg --precision fp64 --nevt 16384 --iterations 4 [--select]

Prints the mean ME, the flat-phase-space estimate of the cross section where it is defined and the throughput.
Also the small driver of the ncu captures whose summaries are under profiles/.
"""
from __future__ import annotations

import argparse
import math

from .me import MatrixElement

GEV2_TO_PB = 0.3893793721e9


def main():
    ap = argparse.ArgumentParser(prog="python -m paper_2503_21935_b200")
    ap.add_argument("--process", default="gg_ttgg", choices=["ee_mumu", "gg_tt", "gg_ttg", "gg_ttgg", "gg_ttggg", "gux_taptamux", "gux_taptamgux",
                                                              "gux_taptamggux"])
    ap.add_argument("--precision", default="fp64", choices=["fp64", "fp32", "mixed"])
    ap.add_argument("--nevt", type=int, default=16384, help="events per iteration (one me_compute call)")
    ap.add_argument("--iterations", type=int, default=4)
    ap.add_argument("--seed", type=int, default=1)
    ap.add_argument("--sqrts", type=float, default=1500.0)
    ap.add_argument("--alphas", type=float, default=0.118, help="<= 0 draws alpha_s ~ U[0.10, 0.13] per event")
    ap.add_argument("--select", action="store_true", help="also draw a helicity and a colour per event")
    ap.add_argument("--device", type=int, default=0)
    a = ap.parse_args()

    import torch
    if not torch.cuda.is_available():
        raise SystemExit("no CUDA device: this library has no CPU path")
    torch.cuda.set_device(a.device)
    m = MatrixElement(a.process, a.precision, device=a.device)
    mom, gs, rh, rc = m.generate(a.nevt, seed=a.seed, sqrts=a.sqrts, alphas=a.alphas)
    mask = m.filter_helicities(mom, gs)
    print(f"{a.process} {a.precision}: {m.npar} particles, {m.ndiag} diagrams, {m.ncol} colour flows, "
          f"{int(mask.sum())} of {m.ncomb} helicities good")
    s_me = s_me2 = s_w = 0.0
    n_tot = 0
    t_gen = t_me = 0.0
    for it in range(a.iterations):
        e0, e1, e2 = (torch.cuda.Event(enable_timing=True) for _ in range(3))
        e0.record()
        mom, gs, rh, rc, wt = m.generate(a.nevt, seed=a.seed, start=it * a.nevt, sqrts=a.sqrts, alphas=a.alphas, want_weight=True)
        e1.record()
        me, sh, sc = m.compute(mom, gs, rh if a.select else None, rc if a.select else None)
        e2.record()
        torch.cuda.synchronize()
        t_gen += e0.elapsed_time(e1) * 1e-3
        t_me += e1.elapsed_time(e2) * 1e-3
        s_me += float(me.sum())
        s_me2 += float((me * me).sum())
        s_w += float((me * wt).sum())
        n_tot += a.nevt
    mean = s_me / n_tot
    err = math.sqrt(max(s_me2 / n_tot - mean * mean, 0.0) / n_tot)
    print(f"events {n_tot}: <ME> = {mean:.9e} +- {err:.2e}")
    # sigma = <ME x RAMBO weight> / (2 s) for massless incoming particles, flat phase space, no cuts
    print(f"flat phase space, no cuts: sigma = {s_w / n_tot / (2.0 * a.sqrts ** 2) * GEV2_TO_PB:.6e} pb")
    if a.select:
        print(f"last iteration: selected helicities {int(sh.min())}..{int(sh.max())}, colours {int(sc.min())}..{int(sc.max())}")
    print(f"throughput: generate {n_tot / max(t_gen, 1e-12):.4e} events/s, matrix elements {n_tot / max(t_me, 1e-12):.4e} MEs/s "
          f"(launch {m.launch_info()})")
    m.close()


if __name__ == "__main__":
    main()
