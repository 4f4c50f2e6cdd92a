#!/usr/bin/env python
"""bench.py -- the driver's measurement contract for the PDF-interpolation hot path.

One "step" = one pass of the hot path over one batch of BASELINE.json configs[2]:
``pdf_xfxq2`` over n queries on the LHAPDF-shaped grid (196 x (6+8+40) knots, 11 flavours,
5 % of the queries extrapolated) followed by ``pdf_alphas_q2`` over the same Q2 array
(a-1 grid layout is one-off and untimed).  The luminosity call
(a-7, configs[4]) and the replica batch (a-8, configs[3]) are timed in the same run under the
same protocol and reported in the ``lumi`` / ``members`` objects of the same JSON line.

metric  = PDF evaluations (points x flavours)/s, whole job (all ranks), inputs resident in HBM.
e2e     = the same metric through ``pdf_xfxq2_host`` + ``pdf_alphas_q2_host`` (pinned HOST
          buffers, H2D and D2H copies inside the timed region).
--impl reference  times the CPU oracle (oracle/) as it stands on the host cores (tier rule).
"""
from __future__ import annotations

import argparse
import json
import os
import subprocess
import sys
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

METRIC = "PDF evaluations (points x flavours)/s"
UNIT = "points*flavours/s"
WORKLOAD = ("configs[2] (C2): 196x(6+8+40) LHAPDF-shaped grid, 11 flavours, "
            "5% of queries extrapolated, + alpha_s over the same Q2 (60 knots)")
# roofline.traffic is a MEASUREMENT, not a constant of this file: dram__bytes_read.sum + dram__bytes_write.sum of
# k_pdf_stream at n = 1e8 (C2) come from the newest ncu capture profiles/*_traffic_pdf_stream_1e8.csv, whose note
# (same name, .md) records the sha256 of the csrc/ tree it was taken on; a capture of another source tree is stale
# and the line carries null (there is no .git on the GPU box, so the tree is identified by content).
# PAPER.md Table 3.3 (L1896-1905), seconds: N_rep -> (LHAPDF CPU, PDFFlow GPU, PDFFlow CPU) on the thesis's system P1
PAPER_TABLE33 = {10: (0.08, 0.07, 0.05), 50: (0.41, 0.35, 0.28), 100: (0.83, 0.69, 0.56),
                 200: (1.87, 1.46, 1.12), 300: (2.85, 1.29, 1.79), 400: (3.63, 1.69, 2.12)}
BYTES_PER_QUERY = 16 + 88          # x, q2 in; 11 fp64 out
BYTES_PER_EVENT = 32 + 8
BYTES_PER_ALPHAS = 16


def parse_args():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=5)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--n", type=int, default=100_000_000, help="queries per GPU and step")
    ap.add_argument("--lumi-n", type=int, default=100_000_000)
    ap.add_argument("--members-n", type=int, default=100_000_000)
    ap.add_argument("--e2e-n", type=int, default=0, help="0 = same as --n")
    ap.add_argument("--cpu-sample", type=int, default=10_000_000)
    ap.add_argument("--path", default="auto", choices=["auto", "direct", "binned"])
    ap.add_argument("--chunk", type=int, default=0, help="binned-path chunk size (0 = library default)")
    ap.add_argument("--table33-reps", type=int, default=10, help="timed calls per N_rep of the Table 3.3 leg (0 = skip)")
    ap.add_argument("--skip-extras", action="store_true", help="only the headline step (no lumi/members/e2e/cpu)")
    return ap.parse_args()


def csrc_sha256():
    """sha256 over the names and contents of the CUDA sources (what a traffic capture is valid for)"""
    import glob
    import hashlib
    h = hashlib.sha256()
    for f in sorted(glob.glob(os.path.join(ROOT, "paper_2302_03343_b200", "csrc", "*"))):
        h.update(os.path.basename(f).encode())
        h.update(open(f, "rb").read())
    return h.hexdigest()


def load_traffic(n):
    """(bytes or None, source dict): the newest profiles/*_traffic_pdf_stream_1e8.csv if it matches this source tree"""
    import csv
    import glob
    import re
    if n != 100_000_000:
        return None, {"traffic_source": None, "traffic_note": "captures exist for n = 1e8 only"}
    caps = sorted(glob.glob(os.path.join(ROOT, "profiles", "*_traffic_pdf_stream_1e8.csv")))
    if not caps:
        return None, {"traffic_source": None, "traffic_note": "no capture under profiles/"}
    cap = caps[-1]
    note = cap[:-4] + ".md"
    want = None
    if os.path.exists(note):
        m = re.search(r"csrc_sha256:\s*([0-9a-f]{64})", open(note).read())
        want = m.group(1) if m else None
    src = {"traffic_source": os.path.relpath(cap, ROOT), "traffic_csrc_sha256": want}
    if want != csrc_sha256():
        src["traffic_note"] = "stale: the capture was taken on another csrc/ tree"
        return None, src
    rd = wr = None
    for row in csv.reader(open(cap)):
        if len(row) > 14 and "k_pdf_stream" in row[4]:
            if row[12] == "dram__bytes_read.sum":
                rd = float(row[14].replace(",", ""))
            if row[12] == "dram__bytes_write.sum":
                wr = float(row[14].replace(",", ""))
    if rd is None or wr is None:
        src["traffic_note"] = "capture unreadable"
        return None, src
    src["traffic_read_bytes"], src["traffic_write_bytes"] = rd, wr
    return rd + wr, src


def load_peaks():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        d = json.load(open(p))
        return float(d["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs)"
    return 6650.0, "fallback (B200_PROFILING.md 6.65 TB/s)"


class ClockSampler:
    """nvidia-smi clocks / throttle reasons DURING the timed region (B200_PROFILING.md recipe)."""
    Q = ("index,clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.active,"
         "clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,"
         "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")

    def __init__(self, index: int):
        self.proc, self.index = None, index
        try:
            self.proc = subprocess.Popen(["nvidia-smi", f"--query-gpu={self.Q}", "--format=csv,noheader,nounits",
                                          "-lms", "100", "-i", str(index)], stdout=subprocess.PIPE,
                                         stderr=subprocess.DEVNULL, text=True)
        except Exception:
            self.proc = None

    def stop(self):
        if self.proc is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        time.sleep(0.15)
        self.proc.terminate()
        try:
            out, _ = self.proc.communicate(timeout=5)
        except Exception:
            self.proc.kill()
            out = ""
        sm, mx, reasons = [], [], set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for line in out.strip().splitlines():
            p = [t.strip() for t in line.split(",")]
            if len(p) < 9:
                continue
            try:
                sm.append(float(p[1])); mx.append(float(p[2]))
            except ValueError:
                continue
            for nm, v in zip(names, p[5:9]):
                if v.lower().startswith("active"):
                    reasons.add(nm)
        sm.sort()
        return {"sm_mhz": sm[len(sm) // 2] if sm else None, "sm_max_mhz": max(mx) if mx else None,
                "reasons": sorted(reasons), "samples": len(sm)}


def run_reference(args):
    """Tier rule: the reference arm is the CPU oracle as it stands, on the host cores, on a bounded
    sample of the same workload per step."""
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    import numpy as np
    import oracle
    from paper_2302_03343_b200 import synth
    spec = synth.grid_c1()
    og = oracle.OracleGrid(spec.x_knots.numpy(), [q.numpy() for q in spec.q2_subgrids], spec.values.numpy(), spec.pids)
    og.set_alphas(spec.alphas_q2.numpy(), spec.alphas_val.numpy())
    n = min(args.cpu_sample, 2_000_000)
    x, q = synth.queries_c2(spec, n)
    x, q = x.numpy(), q.numpy()
    for _ in range(args.warmup):
        og.xfxq2(spec.pids, x[:100_000], q[:100_000])
    t0 = time.perf_counter()
    for _ in range(args.steps):
        og.xfxq2(spec.pids, x, q)
        og.alphas_q2(q)
    dt = time.perf_counter() - t0
    val = n * 11 * args.steps / dt
    line = {"impl": "reference", "metric": METRIC, "value": val, "unit": UNIT, "n_gpus": args.gpus,
            "steps": args.steps, "warmup": args.warmup, "ms_per_step": dt / args.steps * 1e3,
            "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64",
            "data": "synthetic", "config": {"workload": WORKLOAD,
                                            "queries_per_step": n, "l2": "n/a (CPU)"},
            "cpu_baseline": {"value": val, "unit": UNIT, "cores": oracle.num_threads(), "kind": "oracle",
                             "sample": f"first {n} queries of the C2 recipe per step, xfxq2 (11 flavours) + alphas"},
            "e2e": {"value": val, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0}
    print(json.dumps(line))


def timed_steps(torch, dist, world, fn, steps, warmup, sampler_index=None):
    """W untimed + K timed steps, barrier + synchronize on both sides, CUDA events on the launching
    stream, MAX over ranks.  Returns (seconds for K steps, clocks dict, per-kernel profile list)."""
    from paper_2302_03343_b200 import binding
    sampler = ClockSampler(sampler_index) if sampler_index is not None else None
    if sampler is not None:
        time.sleep(1.0)                  # nvidia-smi start-up; its samples then cover warm-up + timed region
    for _ in range(warmup):
        fn()
    torch.cuda.synchronize()
    if world > 1:
        dist.barrier()
    torch.cuda.synchronize()
    binding.pdf_profile_enable(True)
    launches0 = binding.pdf_launch_count()
    a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    a.record()
    for _ in range(steps):
        fn()
    b.record()
    torch.cuda.synchronize()
    if world > 1:
        dist.barrier()
    torch.cuda.synchronize()
    launches = binding.pdf_launch_count() - launches0
    prof = binding.pdf_profile_read(1 << 16)
    binding.pdf_profile_enable(False)
    clocks = sampler.stop() if sampler else None
    ms = a.elapsed_time(b)
    if world > 1:
        t = torch.tensor([ms], dtype=torch.float64, device="cuda")
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
        ms = float(t.item())
    return ms * 1e-3, clocks, prof, launches


def kernel_table(prof, steps):
    """per-kernel: launches per step and total ms per step, from the library's CUDA-event records"""
    agg = {}
    for name, ms in prof:
        c = agg.setdefault(name, [0, 0.0])
        c[0] += 1
        c[1] += ms
    return {k: {"launches_per_step": v[0] / steps, "ms_per_step": v[1] / steps} for k, v in agg.items()}


def roofline_hbm(table, kernels, alg_bytes_per_step, peak_gbs, peak_src, traffic=None):
    """dominant-kernel roofline: algorithmic bytes of the step / summed launch time of `kernels`"""
    ms = sum(table[k]["ms_per_step"] for k in kernels if k in table)
    ach = alg_bytes_per_step / (ms * 1e-3) / 1e9 if ms > 0 else 0.0
    return {"bound": "hbm", "kernel": "+".join(k for k in kernels if k in table), "achieved": ach, "peak": peak_gbs,
            "unit": "GB/s", "frac": ach / peak_gbs, "traffic": traffic, "peak_source": peak_src,
            "kernel_ms_per_step": ms}


def run_ours(args):
    import torch
    import torch.distributed as dist
    from paper_2302_03343_b200 import binding, synth

    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device: the product path has no CPU fallback")
    torch.cuda.set_device(local)
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))
    binding.lib()
    peak_gbs, peak_src = load_peaks()
    pathopt = {"auto": binding.PDF_PATH_AUTO, "direct": binding.PDF_PATH_DIRECT, "binned": binding.PDF_PATH_BINNED}[args.path]

    # ---- headline: configs[2] -------------------------------------------------------------
    spec = synth.grid_c1()
    n = args.n
    g = binding.PdfGrid.from_spec(spec, workspace_for=0 if args.path == "direct" else n)
    g.pdf_grid_set_option(binding.PDF_OPT_PATH, pathopt)
    if args.chunk:
        g.pdf_grid_set_option(binding.PDF_OPT_CHUNK, args.chunk)
        g.attach_workspace(n)
    x, q2 = synth.queries_c2(spec, n, seed=synth.BASE_SEED + 2 + 1000 * rank, device="cuda")
    out = torch.empty((n, 11), dtype=torch.float64, device="cuda")
    aout = torch.empty(n, dtype=torch.float64, device="cuda")

    def step():
        g.pdf_xfxq2(spec.pids, x, q2, out=out)
        g.pdf_alphas_q2(q2, out=aout)

    secs, clocks, prof, launches = timed_steps(torch, dist, world, step, args.steps, args.warmup, sampler_index=local)
    # which kernels the timed pdf_xfxq2 calls took (pdf_alphas_q2 does not touch the record)
    path_taken = {binding.PDF_PATH_DIRECT: "direct", binding.PDF_PATH_BINNED: "binned"}.get(g.pdf_last_path(), "?")
    n_invalid = g.pdf_error_count()
    out_sample = out[:200_000].clone()
    table = kernel_table(prof, args.steps)
    value = world * n * 11 * args.steps / secs
    xf_kernels = [k for k in table if k != "k_alphas"]
    traffic, traffic_src = load_traffic(n) if args.path != "direct" else (None, {"traffic_source": None})
    roof = roofline_hbm(table, xf_kernels, BYTES_PER_QUERY * n, peak_gbs, peak_src, traffic=traffic)
    roof.update(traffic_src)
    roof["algorithmic_bytes"] = BYTES_PER_QUERY * n
    roof["alphas"] = roofline_hbm(table, ["k_alphas"], BYTES_PER_ALPHAS * n, peak_gbs, peak_src)
    line = {"metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps,
            "warmup": args.warmup, "ms_per_step": secs / args.steps * 1e3, "higher_is_better": True,
            "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": {"workload": WORKLOAD,
                       "queries_per_gpu_per_step": n, "path": args.path, "path_taken": path_taken, "n_invalid": n_invalid,
                       "l2": "inputs (1.6 GB) and outputs (9.6 GB) per step exceed the 126 MB L2; no flush needed"},
            "clocks": clocks, "gpu_launches": launches, "kernels": table, "roofline": roof}

    if not args.skip_extras:
        extras(args, torch, dist, world, rank, local, binding, synth, spec, g, x, q2, out, aout, line, peak_gbs, peak_src, out_sample)
    if rank == 0:
        print(json.dumps(line))
    if world > 1:
        dist.destroy_process_group()


def extras(args, torch, dist, world, rank, local, binding, synth, spec, g, x, q2, out, aout, line, peak_gbs, peak_src, out_sample):
    n = args.n
    steps, warm = max(2, min(args.steps, 3)), 3
    # ---- fp64 peak of this device (denominator of the "alu" roofline of pdf_lumi) -------------
    fp64_tf = binding.pdf_measure_fp64_tflops()

    # ---- a-7: luminosity, configs[4] ---------------------------------------------------------
    nl = args.lumi_n
    x1, x2, ql, w = synth.events_c4(nl, seed=synth.BASE_SEED + 4 + 1000 * rank, device="cuda")
    lout = aout[:nl] if nl <= n else torch.empty(nl, dtype=torch.float64, device="cuda")
    if args.path != "direct":
        g.attach_workspace(max(n, nl))
    secs, _, prof, launches = timed_steps(torch, dist, world, lambda: g.pdf_lumi(x1, x2, ql, w, out=lout), steps, warm)
    table = kernel_table(prof, steps)
    lms = sum(v["ms_per_step"] for v in table.values())
    # algorithmic flops/event: 2 stencils x (16 + 11*32) + 2*11 + 2*121 + 22 + weights/logs ~ 1.2 kflop
    flops_event = 1200.0
    ach_tf = flops_event * nl / (lms * 1e-3) / 1e12 if lms else 0.0
    line["lumi"] = {"value": world * nl * steps / secs, "unit": "events/s", "ms_per_step": secs / steps * 1e3,
                    "events_per_gpu_per_step": nl, "gpu_launches": launches, "kernels": table,
                    "roofline": {"bound": "alu", "achieved": ach_tf, "peak": fp64_tf, "unit": "TFLOP/s",
                                 "frac": ach_tf / fp64_tf if fp64_tf else None, "traffic": None,
                                 "peak_source": "pdf_measure_fp64_tflops (independent DFMA chains, this run); "
                                                "nominal 64 DFMA/clk/SM x 148 SMs x 1.965 GHz x 2 = 37.2",
                                 "flops_per_event": flops_event,
                                 "hbm_frac": BYTES_PER_EVENT * nl / (lms * 1e-3) / 1e9 / peak_gbs if lms else None}}
    lumi_sample = (x1[:50_000].cpu().numpy(), x2[:50_000].cpu().numpy(), ql[:50_000].cpu().numpy(),
                   w[:50_000].cpu().numpy(), lout[:50_000].clone().cpu().numpy())
    del x1, x2, ql, w

    # ---- a-8: replica batch, configs[3] (100 members) ------------------------------------------
    nm = args.members_n
    if nm > 0:
        mspec = synth.grid_c1(nmem=100)
        mg = binding.PdfGrid.from_spec(mspec, workspace_for=nm)
        mem = synth.members(mspec, nm, device="cuda")
        secs, _, prof, launches = timed_steps(
            torch, dist, world, lambda: mg.pdf_xfxq2(mspec.pids, x[:nm], q2[:nm], out=out[:nm], member=mem), steps, warm)
        line["members"] = {"value": world * nm * 11 * steps / secs, "unit": UNIT, "ms_per_step": secs / steps * 1e3,
                           "queries_per_gpu_per_step": nm, "nmem": 100, "kernels": kernel_table(prof, steps),
                           "roofline": {"bound": "hbm", "achieved": (BYTES_PER_QUERY + 4) * nm / (secs / steps) / 1e9,
                                        "peak": peak_gbs, "unit": "GB/s",
                                        "frac": (BYTES_PER_QUERY + 4) * nm / (secs / steps) / 1e9 / peak_gbs,
                                        "traffic": None, "peak_source": peak_src,
                                        "note": "whole call (partition + binned kernel + gather), 108 algorithmic B/query"}}
        members_sample = (mspec, x[:50_000].cpu().numpy(), q2[:50_000].cpu().numpy(), mem[:50_000].cpu().numpy(),
                          out[:50_000].clone().cpu().numpy())
        mg.close()
        del mem

    # ---- NEXT-3: Table 3.3 workload: 11 flavours x 2415 x-points x N_rep members ----
    # One pdf_xfxq2_ex call per N_rep (member-major queries, fixed Q2).  Each call is timed alone with CUDA
    # events after an L2 flush (the whole problem would otherwise sit in the 126 MB L2 between repeats).
    table33_sample = None
    if args.table33_reps > 0 and rank == 0:
        tspec = synth.grid_c1(nmem=max(synth.TABLE33_NREP))
        tg = binding.PdfGrid.from_spec(tspec)
        flush = torch.empty(32 * 1024 * 1024, dtype=torch.float64, device="cuda")          # 256 MB > L2
        rows = []
        for nrep in synth.TABLE33_NREP:
            tx, tq, tm = synth.queries_table33(nrep, device="cuda")
            tout = out[: tx.numel()]
            for _ in range(3):
                tg.pdf_xfxq2(tspec.pids, tx, tq, out=tout, member=tm)
            ms = []
            for _ in range(args.table33_reps):
                flush.zero_()
                ea, eb = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
                ea.record()
                tg.pdf_xfxq2(tspec.pids, tx, tq, out=tout, member=tm)
                eb.record()
                torch.cuda.synchronize()
                ms.append(ea.elapsed_time(eb))
            ms.sort()
            med_ex = ms[len(ms) // 2]
            # the structured entry point: the same rows from the 2415 points and the member count
            xg, qg = tx[: synth.TABLE33_NX], tq[: synth.TABLE33_NX]
            tout3 = tout.view(nrep, synth.TABLE33_NX, 11)
            for _ in range(3):
                tg.pdf_xfxq2_xgrid(tspec.pids, xg, qg, nrep, out=tout3)
            ms = []
            for _ in range(args.table33_reps):
                flush.zero_()
                ea, eb = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
                ea.record()
                tg.pdf_xfxq2_xgrid(tspec.pids, xg, qg, nrep, out=tout3)
                eb.record()
                torch.cuda.synchronize()
                ms.append(ea.elapsed_time(eb))
            ms.sort()
            med = ms[len(ms) // 2]
            paper = PAPER_TABLE33[nrep]
            t33_bytes = tx.numel() * 88 + nrep * 4 * 196 * 96 + synth.TABLE33_NX * 16   # rows out + the 4 Q2 rows of every member in
            rows.append({"nrep": nrep, "queries": int(tx.numel()), "ms_median": med, "ms_min": ms[0],
                         "ms_median_xfxq2_ex": med_ex,
                         "value": tx.numel() * 11 / (med * 1e-3), "unit": UNIT,
                         "roofline": {"bound": "hbm", "achieved": t33_bytes / (med * 1e-3) / 1e9, "peak": peak_gbs, "unit": "GB/s",
                                      "frac": t33_bytes / (med * 1e-3) / 1e9 / peak_gbs, "traffic": None, "peak_source": peak_src},
                         "paper_seconds": {"lhapdf_cpu": paper[0], "pdfflow_gpu": paper[1], "pdfflow_cpu": paper[2]}})
            if nrep == max(synth.TABLE33_NREP):
                pick = torch.arange(0, tx.numel(), 31, device="cuda")[:30_000]
                table33_sample = (tspec, tx[pick].cpu().numpy(), tq[pick].cpu().numpy(), tm[pick].cpu().numpy(),
                                  tout[pick].clone().cpu().numpy())
        line["table33"] = {"workload": "Table 3.3: 11 flavours x 2415 fixed x-points x N_rep members at Q2 = 1.65^2 GeV2, "
                                       "C1-shaped 400-member grid (lognormal member noise), member-major queries",
                           "timing": f"median of {args.table33_reps} single calls, CUDA events, 256 MB L2 flush before each",
                           "api": "pdf_xfxq2_xgrid (ms_median, value, roofline); pdf_xfxq2_ex on the member-major expansion (ms_median_xfxq2_ex)",
                           "rows": rows,
                           "paper_hardware": "system P1: i9-9980XE; TITAN V / RTX 2080 Ti (PAPER.md Table 3.2, 3.3): context, not a target"}
        tg.close()
        del flush

    # ---- e2e: host buffers through pdf_xfxq2_host / pdf_alphas_q2_host -------------------------
    ne = args.e2e_n or n
    try:
        hx, hq = x[:ne].cpu().pin_memory(), q2[:ne].cpu().pin_memory()
        hout = torch.empty((ne, 11), dtype=torch.float64).pin_memory()
        haout = torch.empty(ne, dtype=torch.float64).pin_memory()

        def e2e_step():
            g.pdf_xfxq2_host(spec.pids, hx, hq, hout)
            g.pdf_alphas_q2_host(hq, haout)

        e2e_step()
        torch.cuda.synchronize()
        if world > 1:
            dist.barrier()
        t0 = time.perf_counter()
        ksteps = 2
        for _ in range(ksteps):
            e2e_step()
        torch.cuda.synchronize()
        dt = time.perf_counter() - t0
        if world > 1:
            t = torch.tensor([dt], dtype=torch.float64, device="cuda")
            dist.all_reduce(t, op=dist.ReduceOp.MAX)
            dt = float(t.item())
        line["e2e"] = {"value": world * ne * 11 * ksteps / dt, "unit": UNIT, "h2d_bytes_per_step": 16 * ne + 8 * ne,
                       "d2h_bytes_per_step": 88 * ne + 8 * ne, "queries_per_gpu_per_step": ne, "steps": ksteps,
                       "ms_per_step": dt / ksteps * 1e3, "api": "pdf_xfxq2_host + pdf_alphas_q2_host (pinned host tensors)",
                       "checksum": float(torch.nan_to_num(hout[:1000]).sum())}
        del hout, haout
    except Exception as e:  # pinned allocation can fail on a small host
        line["e2e"] = {"value": None, "unit": UNIT, "error": repr(e)}

    # ---- cpu_baseline: the oracle as it stands on the host cores (rank 0, N = 1 only) ----------
    if rank == 0 and world == 1:
        import numpy as np
        import oracle
        ns = min(args.cpu_sample, n)
        og = oracle.OracleGrid(spec.x_knots.numpy(), [q.numpy() for q in spec.q2_subgrids], spec.values.numpy(), spec.pids)
        og.set_alphas(spec.alphas_q2.numpy(), spec.alphas_val.numpy())
        cx, cq = x[:ns].cpu().numpy(), q2[:ns].cpu().numpy()
        t0 = time.perf_counter()
        ref = og.xfxq2(spec.pids, cx, cq)
        og.alphas_q2(cq)
        dt = time.perf_counter() - t0
        line["cpu_baseline"] = {"value": ns * 11 / dt, "unit": UNIT, "cores": oracle.num_threads(), "kind": "oracle",
                                "sample": f"first {ns} queries of this run's C2 batch, xfxq2 (11 flavours) + alphas, {dt:.1f} s"}
        # SURVEY 8(d) "Oracle timing": the whole batch in slices of the sample size (the rows are discarded), and one
        # thread on 1e6 queries (a child process: the OpenMP thread count is fixed when the library loads)
        if n > ns and n <= 200_000_000:
            t0 = time.perf_counter()
            for a0 in range(ns, n, ns):
                sx, sq = x[a0:a0 + ns].cpu().numpy(), q2[a0:a0 + ns].cpu().numpy()
                og.xfxq2(spec.pids, sx, sq)
                og.alphas_q2(sq)
            line["cpu_baseline"]["full_n_seconds"] = dt + time.perf_counter() - t0
            line["cpu_baseline"]["full_n"] = n
        try:
            n1 = min(1_000_000, ns)
            code = ("import sys, time, json; sys.path.insert(0, %r); import oracle\n"
                    "from paper_2302_03343_b200 import synth\n"
                    "spec = synth.grid_c1(); x, q = synth.queries_c2(spec, %d); x, q = x.numpy(), q.numpy()\n"
                    "og = oracle.OracleGrid(spec.x_knots.numpy(), [k.numpy() for k in spec.q2_subgrids], spec.values.numpy(), spec.pids)\n"
                    "og.xfxq2(spec.pids, x[:10000], q[:10000]); t0 = time.perf_counter(); og.xfxq2(spec.pids, x, q); dt = time.perf_counter() - t0\n"
                    "print(json.dumps({'threads': oracle.num_threads(), 'seconds': dt}))") % (ROOT, n1)
            r = subprocess.run([sys.executable, "-c", code], env=dict(os.environ, OMP_NUM_THREADS="1"), capture_output=True,
                               text=True, timeout=300)
            one = json.loads(r.stdout.strip().splitlines()[-1])
            line["cpu_baseline"]["single_thread"] = {"value": n1 * 11 / one["seconds"], "unit": UNIT, "cores": one["threads"],
                                                     "sample": f"{n1} queries of the C2 recipe, xfxq2 (11 flavours), {one['seconds']:.1f} s"}
        except Exception as e:
            line["cpu_baseline"]["single_thread"] = {"value": None, "error": repr(e)}
        # sampled parity at full size, in the timed launch configuration (oracle one by one on the sample)
        import numpy as np
        # the same for the luminosity call (50 000 sampled events of the 1e8 launch)
        og.set_coupling(spec.coupling.numpy())
        lref, ls = og.lumi(*lumi_sample[:4], want_scale=True)
        lerr = np.abs(lumi_sample[4] - lref)
        ltol = oracle.tolerance(lref, ls)
        lok = ~np.isnan(lref)
        line["lumi"]["parity_sample"] = {"n": int(lref.size), "worst_err_over_tol": float(np.max(lerr[lok] / np.maximum(ltol[lok], 1e-300))),
                                         "nan_match": bool(np.array_equal(np.isnan(lumi_sample[4]), ~lok))}
        # and for the replica batch (50 000 sampled queries of the timed launch, 100 members)
        if nm > 0:
            ms_, mx, mq, mm, mgot = members_sample
            mog = oracle.OracleGrid(ms_.x_knots.numpy(), [q.numpy() for q in ms_.q2_subgrids], ms_.values.numpy(), ms_.pids,
                                    nmem=ms_.nmem)
            mref, mS = mog.xfxq2(ms_.pids, mx, mq, member=mm, want_scale=True)
            mok = ~np.isnan(mref)
            mtol = oracle.tolerance(mref, mS)
            line["members"]["parity_sample"] = {"n": int(mx.size), "worst_err_over_tol": float(np.max(np.abs(mgot - mref)[mok] / np.maximum(mtol[mok], 1e-300))),
                                                "nan_match": bool(np.array_equal(np.isnan(mgot), ~mok))}
        # and for the Table 3.3 workload (30 000 sampled rows of the N_rep = 400 call)
        if table33_sample is not None:
            ts_, tx_, tq_, tm_, tgot = table33_sample
            tog = oracle.OracleGrid(ts_.x_knots.numpy(), [q.numpy() for q in ts_.q2_subgrids], ts_.values.numpy(), ts_.pids,
                                    nmem=ts_.nmem)
            tref, tS = tog.xfxq2(ts_.pids, tx_, tq_, member=tm_, want_scale=True)
            ttol = oracle.tolerance(tref, tS)
            line["table33"]["parity_sample"] = {"n": int(tx_.size), "worst_err_over_tol": float(np.max(np.abs(tgot - tref) / np.maximum(ttol, 1e-300))),
                                                "nan_match": bool(not np.isnan(tgot).any() and not np.isnan(tref).any())}
        np_ = min(200_000, ns)
        got = out_sample.cpu().numpy()[:np_]
        _, S = og.xfxq2(spec.pids, cx[:np_], cq[:np_], want_scale=True)
        err = np.abs(got - ref[:np_])
        tol = oracle.tolerance(ref[:np_], S)
        okn = ~np.isnan(ref[:np_])
        aref = np.abs(ref[:np_])
        well = okn & (S[..., 0] <= 100.0 * aref) & (S[..., 1] <= 100.0 * aref) & (aref > 0)       # tests/parity.py STRICT_COND
        line["parity_sample"] = {"n": np_, "worst_err_over_tol": float(np.max(err[okn] / np.maximum(tol[okn], 1e-300))),
                                 "strict_rel_max": float(np.max(err[well] / aref[well])) if well.any() else 0.0,
                                 "strict_rel_max_over": "points with S0, S1 <= 100 |ref| (DESIGN.md C-12)",
                                 "nan_match": bool(np.array_equal(np.isnan(got), ~okn))}


def main():
    args = parse_args()
    if args.impl == "reference":
        run_reference(args)
    else:
        run_ours(args)


if __name__ == "__main__":
    main()
