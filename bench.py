#!/usr/bin/env python
"""bench.py -- MEs/s of the gg -> t tbar g g hot path on B200 (BASELINE.json metric), one JSON line.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--nevt E] [--precision fp64|fp32|mixed]
                    [--process gg_ttgg] [--no-sweep] [--no-extras] [--impl reference]

A "step" is one pass of the whole hot path (me_compute: load, wavefunctions, diagrams, jamps, colour
sum, helicity loop, helicity/colour selection, store) over one batch of seeded RAMBO events.
`value` times the C-ABI call with inputs resident in HBM (CUDA events on the launch stream);
`e2e` times me_compute_host with pinned HOST buffers (H2D + kernels + D2H inside the timed region).
The GPU arm makes its inputs on the device with me_generate (the product's own seeded RAMBO); only the
cpu_baseline leg and --impl reference touch oracle/.
Multi-GPU: events are independent, ranks run replicas on disjoint seeded ranges, no collective on the
data path ("scaling": "weak").  `--gpus N` without a launcher re-executes itself under torchrun.
--impl reference times the CPU oracle.
"""
from __future__ import annotations

import argparse
import json
import os
import re
import subprocess
import sys
import threading
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, ROOT)

from paper_2503_21935_b200.shard import max_over_ranks, rank_range  # noqa: E402

# SURVEY.md 8(d) accounting ("each distinct current once per helicity"): FLOPs of the one-event-per-thread code
PER_HELICITY_ACCOUNTING = {"gg_ttgg": 30331 * 64 + 672}

# FLOPs the kernels EXECUTE per ME according to ncu (thread-level FP64 instruction counts of the committed capture): the
# generator's count is 1.5 % above it for the amplitude kernel, so a fraction from it is printed too
EXECUTED_NCU = {("gg_ttgg", "fp64"): {"flops_per_me": 861206 + 64 * 1202 + 1080, "source": "profiles/r2_gg_ttgg_fp64_pipeline_ncu_full.txt: "
                                      "amplitude kernel 1.411e10 FP64 FLOP / 16384 events = 861206 (generator: 875584); colour and setup kernels as the generator counts them"}}

METRIC = "matrix elements/sec (MEs/s) for gg->ttbar gg fp64 & fp32 on 1 B200; % of FMA peak"
UNIT = "MEs/s"
ALPHAS = {"ee_mumu": 0.118, "gg_tt": 0.118, "gg_ttg": 0.118, "gg_ttgg": None, "gg_ttggg": 0.118, "gux_taptamux": None, "gux_taptamgux": None,
          "gux_taptamggux": None}
DTYPE = {"fp64": "f64", "fp32": "f32", "mixed": "f64+f32"}
GROUP = ("gg_ttgg", "gg_ttggg")   # lane-group pipeline: colour contraction on the tensor cores


def parse():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=10)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--nevt", type=int, default=1 << 20, help="events per step (per GPU)")
    ap.add_argument("--process", default="gg_ttgg")
    ap.add_argument("--precision", default="fp64", choices=["fp64", "fp32", "mixed"])
    ap.add_argument("--impl", default="b200", choices=["b200", "reference"])
    ap.add_argument("--no-sweep", action="store_true", help="skip the events-per-launch sweep 2^8..2^22")
    ap.add_argument("--no-extras", action="store_true", help="skip fp32/mixed lines, cpu_baseline and e2e")
    ap.add_argument("--multichannel-only", action="store_true",
                    help="only the me_compute_multichannel leg (the command of the ncu capture of the diagram kernel)")
    return ap.parse_args()


def flops_per_me(process, ngood):
    """Algorithmic FLOPs per ME of the generated code (FMA = 2), counted by the generator (gen/flops.json):
    (all, the part that runs on the FMA pipes when the colour contraction is on the tensor cores, detail)."""
    path = os.path.join(ROOT, "paper_2503_21935_b200", "csrc", "gen", "flops.json")
    with open(path) as f:
        d = json.load(f)[process]
    allf = d["per_event"] + ngood * d["per_helicity"]
    return allf, d["per_event"] + ngood * d["amplitudes_per_helicity"], d


def profile_traffic(process, precision):
    """DRAM bytes per event of the dominant kernel (amplitude kernel of the pipeline, or the event kernel) from the
    committed ncu summary of this build, or None: (dram__bytes_read.sum + dram__bytes_write.sum) / events of the
    captured launch."""
    for kind, kernel in (("pipeline", "amp_kernel"), ("event", "event_kernel")):
        path = os.path.join(ROOT, "profiles", f"r2_{process}_{precision}_{kind}_ncu_full.txt")
        if not os.path.exists(path):
            continue
        txt = open(path).read()
        m = re.search(r"# events per captured (?:amplitude )?launch: (\d+)", txt)
        for b in txt.split("\nKernel Name"):
            if kernel not in b.split("\n")[0]:
                continue
            tot = 0.0
            for key in ("dram__bytes_read.sum", "dram__bytes_write.sum"):
                mm = re.search(re.escape(key) + r" \[(\w+)\] = ([0-9.eE+-]+)", b)
                if not mm:
                    return None, None
                tot += float(mm.group(2)) * {"byte": 1, "Kbyte": 1e3, "Mbyte": 1e6, "Gbyte": 1e9}[mm.group(1)]
            if m:
                return tot / int(m.group(1)), os.path.relpath(path, ROOT)
    return None, None


class ClockSampler:
    """nvidia-smi clocks / throttle reasons sampled DURING the timed region (B200_PROFILING.md)."""

    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,"
         "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")

    def __init__(self, index):
        self.index, self.rows, self.proc = index, [], None

    def __enter__(self):
        try:
            self.proc = subprocess.Popen(["nvidia-smi", f"--id={self.index}", f"--query-gpu={self.Q}", "--format=csv,noheader,nounits",
                                          "-lms", "100"], stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            self.t = threading.Thread(target=self._read, daemon=True)
            self.t.start()
        except OSError:
            self.proc = None
        return self

    def _read(self):
        for line in self.proc.stdout:
            self.rows.append([x.strip() for x in line.split(",")])

    def __exit__(self, *a):
        if self.proc:
            time.sleep(0.15)
            self.proc.terminate()
            self.t.join(timeout=2)

    def summary(self):
        sm, mx, reasons, pw = [], [], set(), []
        for r in self.rows:
            try:
                sm.append(float(r[0])); mx.append(float(r[1])); pw.append(float(r[2]))
            except (ValueError, IndexError):
                continue
            for name, v in zip(("hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"), r[3:7]):
                if v.lower().startswith("active"):
                    reasons.add(name)
        if not sm:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["unavailable"]}
        return {"sm_mhz": float(np.median(sm)), "sm_max_mhz": float(max(mx)), "power_w_max": float(max(pw)),
                "samples": len(sm), "reasons": sorted(reasons)}


def time_device(torch, m, bufs, steps, warmup, select=True):
    """ms per step of me_compute with device-resident inputs: CUDA events on the launch stream."""
    mom, gs, rh, rc, out, sh, sc = bufs
    stream = torch.cuda.current_stream()
    kw = dict(out=out, selhel=sh if select else None, selcol=sc if select else None, stream=stream)
    for _ in range(warmup):
        m.compute(mom, gs, rh if select else None, rc if select else None, **kw)
    torch.cuda.synchronize()
    ev = [torch.cuda.Event(enable_timing=True) for _ in range(steps + 1)]
    ev[0].record(stream)
    for k in range(steps):
        m.compute(mom, gs, rh if select else None, rc if select else None, **kw)
        ev[k + 1].record(stream)
    torch.cuda.synchronize()
    per = [ev[k].elapsed_time(ev[k + 1]) for k in range(steps)]
    return ev[0].elapsed_time(ev[steps]), per


def oracle_inputs(process, nevt, seed=1, start=0):
    from oracle import rambo as R
    return (R.make_momenta(process, nevt, seed=seed, start=start), R.make_gs(nevt, seed=seed, alphas=ALPHAS[process], start=start))


def cpu_baseline(process, seconds_target=15.0):
    """The oracle as it stands, on this box's host cores, on a bounded sample of the same workload, and the
    oracle's own count of FLOPs per ME ("counted mode": the same source compiled with an operation-counting scalar)."""
    from oracle import oracle as O
    n0 = {"ee_mumu": 16384, "gg_tt": 16384, "gg_ttg": 4096, "gg_ttgg": 256, "gg_ttggg": 16, "gux_taptamggux": 2048}.get(process, 16384)
    mom, gs = oracle_inputs(process, n0)
    O.me(process, mom[:8], gs[:8])
    t = time.perf_counter(); O.me(process, mom, gs); dt = time.perf_counter() - t
    n = int(max(n0, min(1 << 20, n0 * seconds_target / max(dt, 1e-3))))
    mom, gs = oracle_inputs(process, n)
    mask = O.good_helicities(process, mom[:n0], gs[:n0])
    t = time.perf_counter(); O.me(process, mom, gs, mask=mask); dt = time.perf_counter() - t
    cnt = O.count_ops(process, mom[0], float(gs[0]), mask=mask)
    return {"value": n / dt, "unit": UNIT, "cores": O.num_threads(), "kind": "oracle",
            "sample": f"first {n} events of the seeded {process} stream (seed 1), good helicities only, {dt:.1f} s",
            "flops_per_me_counted": cnt["flops"],
            "flops_note": "oracle/me_oracle.cpp compiled with its operation-counting scalar (-DORC_COUNT): additions + "
                          "multiplications + divisions + square roots of one event over the good helicities (every diagram, "
                          "4x4 matrices, each distinct current once per helicity, colour sum as the plain double sum)"}


# The other BASELINE.json configs and the Table-4 process, at their sizes: timed in the
# default run on rank 0 and reported under "configs" (the headline line stays gg_ttgg = C4)
CONFIGS = (("ee_mumu", 16384, ("fp64",)), ("gg_tt", 524288, ("fp64", "fp32")), ("gg_ttg", 524288, ("fp64", "fp32", "mixed")),
           ("gg_ttggg", 262144, ("fp64", "fp32", "mixed")), ("gux_taptamggux", 524288, ("fp64", "fp32", "mixed")))


def bench_configs(torch, MatrixElement, local, peaks, nominal, steps=10, warmup=3):
    """MEs/s and roofline fraction of every (process, precision) of CONFIGS: me_compute with selection on, inputs made on
    the device, CUDA events on the launch stream, clocks sampled during each timed region."""
    res = {}
    for proc, n, precs in CONFIGS:
        gen = MatrixElement(proc, "fp64", device=local)
        mom, gs, rh, rc = gen.generate(n, seed=1, alphas=0.0 if ALPHAS[proc] is None else ALPHAS[proc])
        gen.close()
        dev = mom.device
        bufs = (mom, gs, rh, rc, torch.empty(n, dtype=torch.float64, device=dev),
                torch.empty(n, dtype=torch.int32, device=dev), torch.empty(n, dtype=torch.int32, device=dev))
        res[proc] = {}
        for prec in precs:
            m = MatrixElement(proc, prec, device=local)
            mask = m.filter_helicities(mom, gs)
            torch.cuda.synchronize()
            with ClockSampler(local) as cs:
                _, per = time_device(torch, m, bufs, steps, warmup)
            info = m.launch_info()
            m.close()
            ms = float(np.mean(per))
            ngood = int(mask.sum())
            fl_all, fl_fma, _ = flops_per_me(proc, ngood)
            on_tensor = proc in GROUP and prec != "fp64"
            fl = fl_fma if on_tensor else fl_all
            pipe = "fp32" if prec == "fp32" else "fp64"
            ach = fl * n / (ms * 1e-3) * 1e-12
            res[proc][prec] = {"value": n / (ms * 1e-3), "unit": UNIT, "ms_per_step": ms, "nevt": n, "steps": steps, "warmup": warmup,
                               "good_helicities": ngood, "flops_per_me": fl, "tflops": ach, "roofline_frac": ach / peaks[pipe],
                               "roofline_frac_nominal": ach / nominal[pipe], "colour_on_tensor_cores": on_tensor,
                               "clocks": cs.summary(), "launch": info}
    return res


def bench_multichannel(torch, MatrixElement, local, process="gg_ttgg", n=65536, steps=10, warmup=3):
    """me_compute_multichannel (reading R17): events of random channels in one call, fp64."""
    m = MatrixElement(process, "fp64", device=local)
    mom, gs, rh, rc = m.generate(n, seed=1, alphas=0.0 if ALPHAS[process] is None else ALPHAS[process])
    m.filter_helicities(mom, gs)
    chan = torch.randint(0, m.ndiag, (n,), dtype=torch.int32, device=mom.device, generator=torch.Generator(device=mom.device).manual_seed(1))
    stream = torch.cuda.current_stream()
    for _ in range(warmup):
        m.compute_multichannel(mom, gs, chan, rh, rc)
    torch.cuda.synchronize()
    e0, e1, e2 = (torch.cuda.Event(enable_timing=True) for _ in range(3))
    e0.record(stream)
    for _ in range(steps):
        m.compute_multichannel(mom, gs, chan, rh, rc)
    e1.record(stream)
    sh, sc = (torch.empty(n, dtype=torch.int32, device=mom.device) for _ in range(2))
    out = torch.empty(n, dtype=torch.float64, device=mom.device)
    for _ in range(steps):
        m.compute(mom, gs, rh, rc, out=out, selhel=sh, selcol=sc)
    e2.record(stream)
    torch.cuda.synchronize()
    t_mc, t_me = e0.elapsed_time(e1) / steps, e1.elapsed_time(e2) / steps
    m.close()
    return {"workload": process, "nevt": n, "value": n / (t_mc * 1e-3), "unit": UNIT, "ms_per_step": t_mc,
            "me_compute_ms_per_step_same_batch": t_me, "diagram_kernel_share": max(0.0, 1.0 - t_me / t_mc),
            "api": "me_compute_multichannel: me_compute + the diagram-by-diagram kernel for num / den, random channels in one call"}


def run_reference(a):
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    from oracle import oracle as O
    process = a.process
    n0 = {"ee_mumu": 16384, "gg_tt": 16384, "gg_ttg": 16384, "gg_ttgg": 8192, "gg_ttggg": 64, "gux_taptamggux": 16384}.get(process, 16384)
    mom, gs = oracle_inputs(process, n0)
    mask = O.good_helicities(process, mom[: min(n0, 256)], gs[: min(n0, 256)])
    for _ in range(a.warmup):
        O.me(process, mom[: max(8, n0 // 8)], gs[: max(8, n0 // 8)], mask=mask)
    t = time.perf_counter()
    for _ in range(a.steps):
        O.me(process, mom, gs, mask=mask)
    dt = time.perf_counter() - t
    val = a.steps * n0 / dt
    sample = f"each step = first {n0} events of the seeded {process} stream (bounded sample of the {a.nevt}-event workload)"
    print(json.dumps({
        "impl": "reference", "metric": METRIC, "value": val, "unit": UNIT, "n_gpus": a.gpus, "steps": a.steps,
        "warmup": a.warmup, "ms_per_step": 1e3 * dt / a.steps, "higher_is_better": True, "scaling": "weak",
        "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": {"workload": process, "events_per_step_per_gpu": a.nevt, "precision": "fp64",
                   "inputs": "seeded RAMBO sqrt(s)=1500 GeV, alpha_s~U[0.10,0.13]", "reference_events_per_step": n0},
        "cpu_baseline": {"value": val, "unit": UNIT, "cores": O.num_threads(), "kind": "oracle", "sample": sample},
        "e2e": {"value": val, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0}))


def respawn_under_torchrun(a):
    """`python bench.py --gpus N` without a launcher: run the same command as N ranks on this node."""
    import socket
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        port = s.getsockname()[1]
    cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", f"--nproc-per-node={a.gpus}", "--master-addr", "127.0.0.1",
           "--master-port", str(port), os.path.abspath(__file__)] + sys.argv[1:]
    sys.exit(subprocess.call(cmd))


def main():
    a = parse()
    if a.gpus > 1 and "WORLD_SIZE" not in os.environ:
        return respawn_under_torchrun(a)
    if a.impl == "reference":
        return run_reference(a)
    import torch
    import torch.distributed as dist

    from paper_2503_21935_b200.me import MatrixElement, fma_peak, mma_peak

    if a.multichannel_only:
        print(json.dumps(bench_multichannel(torch, MatrixElement, 0, process=a.process, steps=a.steps, warmup=a.warmup)))
        return
    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))
    torch.cuda.set_device(local)
    dev = torch.device("cuda", local)
    process, nevt = a.process, a.nevt
    extras = rank == 0 and not a.no_extras

    def barrier(sync_ranks):
        if sync_ranks and world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    # seeded inputs made on the device: rank r takes events [r*nevt, (r+1)*nevt) of the stream (disjoint shards, no
    # exchange); rank 0 makes up to 2^22 events when it also runs the events-per-launch sweep
    sweep = extras and not a.no_sweep and process == "gg_ttgg"
    start, _ = rank_range(nevt, rank, world)
    nmax = max(nevt, 1 << 22) if sweep else nevt
    gen = MatrixElement(process, "fp64", device=local)
    alphas_dev = 0.0 if ALPHAS[process] is None else ALPHAS[process]
    mom_all, gs_all, rh_all, rc_all = gen.generate(nmax, seed=1, start=start, alphas=alphas_dev)
    torch.cuda.synchronize()
    gen.close()
    out_all = torch.empty(nmax, dtype=torch.float64, device=dev)
    sh_all = torch.empty(nmax, dtype=torch.int32, device=dev)
    sc_all = torch.empty(nmax, dtype=torch.int32, device=dev)
    big = (mom_all, gs_all, rh_all, rc_all, out_all, sh_all, sc_all)
    bufs = tuple(x[:nevt] for x in big)

    def bench_precision(prec, steps, warmup, sync_ranks):
        m = MatrixElement(process, prec, device=local)
        mask = m.filter_helicities(bufs[0], bufs[1])
        barrier(sync_ranks)
        with ClockSampler(local) as cs:
            total_ms, per = time_device(torch, m, bufs, steps, warmup)
        barrier(sync_ranks)
        info = m.launch_info()
        return m, mask, total_ms, per, cs.summary(), info

    m, mask, total_ms, per, clocks, info = bench_precision(a.precision, a.steps, a.warmup, True)
    total_ms = max_over_ranks(total_ms, dist if world > 1 else None, dev)
    ms_per_step = total_ms / a.steps
    value = world * nevt / (ms_per_step * 1e-3)
    ngood = int(mask.sum())
    fl_all, fl_fma, fl_detail = flops_per_me(process, ngood)
    on_tensor = process in GROUP and a.precision != "fp64"   # colour contraction off the FMA pipes
    bytes_per_event = m.npar * 32 + 8 + 16 + 16
    line = {
        "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": a.steps, "warmup": a.warmup,
        "ms_per_step": ms_per_step, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
        "dtype": DTYPE[a.precision], "data": "synthetic",
        "config": {"workload": process, "events_per_step_per_gpu": nevt, "precision": a.precision,
                   "inputs": "seeded RAMBO sqrt(s)=1500 GeV made on the device (me_generate), alpha_s~U[0.10,0.13], "
                             "helicity+colour selection on",
                   "l2": "momenta+randoms+outputs per step = %.0f MB %s the 126 MB L2; the path is FMA-bound (%d B per "
                         "event against ~%.2g FLOP), no flush applied" % (nevt * bytes_per_event / 1e6,
                                                                           ">" if nevt * bytes_per_event > 126e6 else "<",
                                                                           bytes_per_event, fl_all),
                   "good_helicities": ngood, "launch": info, "parallelism": f"replicas x{world}"},
        "clocks": clocks, "gpu_launches": a.steps * max(1, info.get("launches", 1)),
    }
    if rank == 0:
        prec_peak = "fp32" if a.precision == "fp32" else "fp64"
        with ClockSampler(local) as cs_peak:
            peak = fma_peak(prec_peak, local)
            for _ in range(3):   # a few more runs so that the sampler sees the microbenchmark under load
                peak = max(peak, fma_peak(prec_peak, local))
        # the FP64 units serve DFMA and DMMA alike: the measured peak of the pipe is the higher of the two microbenchmarks
        peak_chain, peak_dmma = peak, (mma_peak("dmma", local) if prec_peak == "fp64" else None)
        if peak_dmma is not None:
            peak = max(peak_chain, peak_dmma)
        props = torch.cuda.get_device_properties(local)
        max_mhz = clocks.get("sm_max_mhz") or 1965.0
        nominal = props.multi_processor_count * (64 if prec_peak == "fp64" else 128) * 2 * max_mhz * 1e-6
        step_ms = float(np.mean(per))
        fl = fl_fma if on_tensor else fl_all
        achieved = fl * nevt / (step_ms * 1e-3) * 1e-12
        tr, tr_src = profile_traffic(process, a.precision)
        line["roofline"] = {
            "bound": "alu", "achieved": achieved, "peak": peak, "unit": "TFLOP/s", "frac": achieved / peak,
            "frac_nominal": achieved / nominal, "nominal_peak": nominal,
            "nominal_peak_source": f"{props.multi_processor_count} SMs x {64 if prec_peak == 'fp64' else 128} lanes x 2 x "
                                   f"{max_mhz:.0f} MHz (device properties, nvidia-smi clocks.max.sm)",
            "kernel": ("the whole step (setup + amplitude + colour kernels of every chunk); the amplitude kernel is the "
                       "dominant one, its share of the step is in profiles/ (ncu launch list)") if process in GROUP else "event_kernel",
            "step_ms": step_ms, "flops_per_me": fl,
            "flops_source": "generator count of the operations the kernels execute (FMA = 2, DESIGN.md section 5): "
                            f"{fl_detail['amplitudes_per_helicity']} (amplitudes) + {fl_detail['colour_per_helicity']} (colour sum, "
                            f"symmetric half) per helicity x {ngood} good helicities + {fl_detail['per_event']} per event"
                            + ("; the colour contraction of this build runs on the TF32 tensor cores, so only the "
                               "amplitude part is credited against the FMA peak" if on_tensor else ""),
            "frac_all_flops": fl_all * nevt / (step_ms * 1e-3) * 1e-12 / peak,
            "flops_per_me_executed_ncu": (EXECUTED_NCU.get((process, a.precision))),
            "frac_executed_ncu": (EXECUTED_NCU[(process, a.precision)]["flops_per_me"] * nevt / (step_ms * 1e-3) * 1e-12 / peak
                                  if (process, a.precision) in EXECUTED_NCU else None),
            "tensor_flops_per_me": (fl_all - fl_fma) if on_tensor else 0,
            "peak_source": (f"max of me_fma_peak(fp64) = {peak_chain:.2f} (register-resident DFMA chains, best of 4) and "
                            f"me_mma_peak(dmma) = {peak_dmma:.2f} (DMMA m8n8k4 runs on the same FP64 units), measured on this GPU in this run"
                            if peak_dmma is not None else
                            f"me_fma_peak({prec_peak}): register-resident FMA chains measured on this GPU in this run (best of 4)"),
            "peak_fma_chain": peak_chain,
            "peak_clocks": cs_peak.summary(),
            "traffic": (tr * nevt if tr is not None else None),
            "traffic_source": tr_src,
            "traffic_note": "DRAM bytes of the dominant kernel per step, scaled per event from the ncu capture named in "
                            "traffic_source; the path is FMA-bound, not HBM-bound",
            "tensor_peaks": ({"dmma_m8n8k4_f64": mma_peak("dmma", local), "tf32_m16n8k8": mma_peak("tf32", local),
                              "note": "me_mma_peak, measured in this run; the colour contraction (K2) uses DMMA in the fp64 build "
                                      "(same FP64 units as DFMA: fewer issue slots, no extra throughput) and 2xTF32 in fp32/mixed"}
                             if process in GROUP else None),
            "frac_per_helicity_accounting": (PER_HELICITY_ACCOUNTING[process] * nevt / (step_ms * 1e-3) * 1e-12 / peak
                                             if process in PER_HELICITY_ACCOUNTING and not on_tensor else None),
        }
    m.close()
    if extras:
        # e2e: host buffers (pinned) -> me_compute_host -> host results
        pin = lambda x: x.cpu().pin_memory()
        hm, hg, hr, hc = (pin(x) for x in bufs[:4])
        ho = torch.empty(nevt, dtype=torch.float64).pin_memory()
        hsh = torch.empty(nevt, dtype=torch.int32).pin_memory()
        hsc = torch.empty(nevt, dtype=torch.int32).pin_memory()
        m = MatrixElement(process, a.precision, device=local)
        m.set_good_helicities(mask)
        for _ in range(max(1, a.warmup)):
            m.compute_host(hm, hg, hr, hc, out=ho, selhel=hsh, selcol=hsc)
        t0 = time.perf_counter()
        for _ in range(a.steps):
            m.compute_host(hm, hg, hr, hc, out=ho, selhel=hsh, selcol=hsc)
        dt = time.perf_counter() - t0
        m.close()
        line["e2e"] = {"value": a.steps * nevt / dt, "unit": UNIT,
                       "h2d_bytes_per_step": int(sum(x.numel() * x.element_size() for x in (hm, hg, hr, hc))),
                       "d2h_bytes_per_step": int(nevt * 16),
                       "api": "me_compute_host (pinned host buffers; chunks double-buffered over copy-in / compute / copy-out streams)"}
        del hm, hg, hr, hc, ho, hsh, hsc
        others = {}
        for prec in ("fp64", "fp32", "mixed"):
            if prec == a.precision:
                continue
            m2, mk2, tot2, per2, clk2, info2 = bench_precision(prec, a.steps, a.warmup, False)
            ms2 = float(np.mean(per2))
            pk = fma_peak("fp32", local) if prec == "fp32" else max(fma_peak("fp64", local), mma_peak("dmma", local))
            ot = process in GROUP and prec != "fp64"
            ach = (fl_fma if ot else fl_all) * nevt / (ms2 * 1e-3) * 1e-12
            others[prec] = {"value": nevt / (ms2 * 1e-3), "unit": UNIT, "ms_per_step": ms2, "launch": info2,
                            "roofline_frac": ach / pk, "roofline_frac_all_flops": fl_all * nevt / (ms2 * 1e-3) * 1e-12 / pk,
                            "peak_tflops": pk, "clocks": clk2}
            m2.close()
        line["other_precisions"] = others
        if sweep:
            sw = {}
            for prec in ("fp64", "fp32", "mixed"):
                m3 = MatrixElement(process, prec, device=local)
                m3.set_good_helicities(mask)
                for lg in range(8, 23):
                    n = 1 << lg
                    b3 = tuple(x[:n] for x in big)
                    tot3, per3 = time_device(torch, m3, b3, 10, 3)
                    sw[f"{prec}:{n}"] = n / (float(np.median(per3)) * 1e-3)
                m3.close()
            line["sweep_mes_per_s"] = sw
            line["sweep_note"] = "median of 10 launches per point, events per launch 2^8 .. 2^22"
            line["sweep_best"] = {p: max((v, k) for k, v in sw.items() if k.startswith(p))[1] for p in ("fp64", "fp32", "mixed")}
        # self-contained step: inputs made on the device by me_generate, then me_compute
        m4 = MatrixElement(process, a.precision, device=local)
        m4.set_good_helicities(mask)
        stream = torch.cuda.current_stream()
        for _ in range(a.warmup):
            g = m4.generate(nevt, seed=1, alphas=alphas_dev)
            m4.compute(*g, out=bufs[4], selhel=bufs[5], selcol=bufs[6])
        torch.cuda.synchronize()
        e0, e1, e2 = (torch.cuda.Event(enable_timing=True) for _ in range(3))
        e0.record(stream)
        for _ in range(a.steps):
            g = m4.generate(nevt, seed=1, alphas=alphas_dev)
        e1.record(stream)
        for _ in range(a.steps):
            g = m4.generate(nevt, seed=1, alphas=alphas_dev)
            m4.compute(*g, out=bufs[4], selhel=bufs[5], selcol=bufs[6])
        e2.record(stream)
        torch.cuda.synchronize()
        line["device_inputs"] = {"generate_events_per_s": a.steps * nevt / (e0.elapsed_time(e1) * 1e-3),
                                 "generate_plus_compute_mes_per_s": a.steps * nevt / (e1.elapsed_time(e2) * 1e-3),
                                 "api": "me_generate (seeded RAMBO on the device) + me_compute"}
        m4.close()
        if process == "gg_ttgg" and nevt == 1 << 20:   # the default run only
            max_mhz = clocks.get("sm_max_mhz") or 1965.0
            sms = torch.cuda.get_device_properties(local).multi_processor_count
            peaks = {"fp64": max(fma_peak("fp64", local), mma_peak("dmma", local)), "fp32": fma_peak("fp32", local)}
            nominal = {"fp64": sms * 64 * 2 * max_mhz * 1e-6, "fp32": sms * 128 * 2 * max_mhz * 1e-6}
            line["configs"] = bench_configs(torch, MatrixElement, local, peaks, nominal)
            line["configs_note"] = ("BASELINE.json configs C1-C3, C5 and the Table-4 process at their sizes, 10 timed steps each after 3 "
                                    "warm-ups, selection on; roofline_frac against the measured peaks %s TFLOP/s (fp64 = max of DFMA "
                                    "chain and DMMA), roofline_frac_nominal against %s; fp32 / mixed of the lane-group processes credit "
                                    "the amplitude FLOPs only (colour contraction on the TF32 tensor cores)"
                                    % ({k: round(v, 2) for k, v in peaks.items()}, {k: round(v, 2) for k, v in nominal.items()}))
            line["multichannel"] = bench_multichannel(torch, MatrixElement, local)
        cb = cpu_baseline(process)
        line["roofline"]["flops_per_me_oracle"] = cb.pop("flops_per_me_counted")
        line["roofline"]["flops_per_me_oracle_note"] = cb.pop("flops_note")
        line["cpu_baseline"] = cb
    if rank == 0:
        print(json.dumps(line))
    if world > 1:
        dist.barrier()
        dist.destroy_process_group()


if __name__ == "__main__":
    main()
