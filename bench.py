#!/usr/bin/env python
"""bench.py -- throughput of the HEALPix SHT hot path on B200, one JSON line.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--workload cfg5] [--impl ours|reference]

A "step" is one pass of the whole hot path over one batch: map2alm + alm2map + alm2map_adjoint + map2alm_adjoint
(SURVEY 8(a) rows a1, a3, s1, s2, d1, d2), i.e. 4 * batch transforms.  Default workload: BASELINE configs[4]
(nside 4096, lmax = mmax = 8191, batch 1, fp64), the largest configuration the metric is quoted on.
`value` is device-timed (two CUDA events around K back-to-back steps of the four public calls) with the inputs
resident in HBM; `e2e` goes through the same calls with pinned HOST buffers and the host<->device copies inside the
timed region; the per-stage times behind `roofline` come from a separate, instrumented pass over the stage-level
entry points.  N > 1 runs one independent replica per GPU (batch channels are independent: no data-path collective;
DESIGN.md "Multi-GPU"); launched without torchrun, `--gpus N` spawns the N ranks itself.
"""
from __future__ import annotations

import argparse
import json
import os
import subprocess
import sys
import tempfile
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

import numpy as np  # noqa: E402

from paper_2510_01785_b200 import replicas, synth  # noqa: E402

METRIC = "map2alm/alm2map transforms/s at Nside 1024\u20134096; % of FP64/HBM roofline"  # byte-identical to BASELINE.json
UNIT = "transforms/s"
# B200 plain-ALU peaks: 148 SMs x 64 (128) FP64 (FP32) FMA lanes x 2 flop x 1.965 GHz
PEAK_TFLOPS = {"f64": 148 * 64 * 2 * 1.965e9 / 1e12, "f32": 148 * 128 * 2 * 1.965e9 / 1e12}


def load_peaks():
    path = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(path):
        with open(path) as f:
            return json.load(f).get("hbm_gbs", 6650.0), "measured"
    return 6650.0, "fallback"


def oracle_sample_rings(nside, count):
    """`count` rings spread over the sphere (caps and belt), 1-based."""
    nr = 4 * nside - 1
    return sorted(set(1 + int((k + 0.5) * nr / count) for k in range(count)))


def oracle_cost_fraction(nside, lmax, mmax, rings):
    """Share of one alm2map the oracle spends on `rings`: its operation count per ring is nalm + N_ring (mmax+1)."""
    nalm = synth.alm_count(lmax, mmax)

    def npix_ring(r):
        i = min(r, 4 * nside - r)
        return 4 * i if i < nside else 4 * nside

    tot = sum(nalm + npix_ring(r) * (mmax + 1) for r in range(1, 4 * nside))
    return sum(nalm + npix_ring(r) * (mmax + 1) for r in rings) / tot


def run_reference(args, cfg):
    """--impl reference: the CPU oracle, as it stands, on the host cores (rank 0 only)."""
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    import oracle

    nside, lmax, mmax, batch = cfg["nside"], cfg["lmax"], cfg["mmax"], cfg["batch"]
    cores = oracle.num_threads()
    alm = synth.powerlaw_alm(cfg["seed"], lmax, mmax, 1)[0]
    if cfg["dtype"] == "f32":
        alm = alm.astype(np.complex64).astype(np.complex128)
    nr = max(2, cores // 2) if nside >= 1024 else 4 * nside - 1
    rings = oracle_sample_rings(nside, nr)
    frac = oracle_cost_fraction(nside, lmax, mmax, rings)
    for _ in range(args.warmup if nside < 1024 else min(args.warmup, 1)):
        oracle.alm2map_rings(nside, lmax, mmax, alm, rings)
    t0 = time.perf_counter()
    for _ in range(args.steps):
        oracle.alm2map_rings(nside, lmax, mmax, alm, rings)
    dt = time.perf_counter() - t0
    value = frac * args.steps / dt  # transforms / s
    sample = (f"alm2map on {len(rings)} of {4 * nside - 1} rings = {frac:.3e} of one transform per step "
              f"(share of the oracle's own operation count), long double, OpenMP over rings")
    line = {
        "impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
        "warmup": args.warmup, "ms_per_step": 1e3 * dt / args.steps, "higher_is_better": True, "scaling": "weak",
        "vs_baseline": None, "dtype": "f80", "data": "synthetic",
        "config": {"workload": workload_name(cfg), "sample": sample},
        "cpu_baseline": {"value": value, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": sample},
        "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
    }
    print(json.dumps(line), flush=True)


def workload_name(cfg):
    return (f"BASELINE configs[{cfg['index']}]: nside={cfg['nside']} RING lmax=mmax={cfg['lmax']} batch={cfg['batch']} "
            f"{cfg['dtype']}")


class ClockSampler:
    """nvidia-smi clocks / throttle reasons DURING the timed region (B200_PROFILING.md recipe)."""

    FIELDS = ("index,clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.active,clocks_event_reasons.hw_slowdown,"
              "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
              "clocks_event_reasons.sw_power_cap")

    def __init__(self, gpu_index):
        self.gpu = gpu_index
        self.proc = None
        self.path = None

    def start(self):
        try:
            fd, self.path = tempfile.mkstemp(suffix=".csv")
            os.close(fd)
            self.proc = subprocess.Popen(
                ["nvidia-smi", f"--query-gpu={self.FIELDS}", "--format=csv,noheader,nounits", "-lms", "100", "-i",
                 str(self.gpu)], stdout=open(self.path, "w"), stderr=subprocess.DEVNULL)
        except Exception:
            self.proc = None

    def count(self):
        try:
            with open(self.path) as f:
                return sum(1 for _ in f)
        except Exception:
            return 0

    def stop(self):
        out = {"sm_mhz": None, "sm_max_mhz": None, "reasons": [], "samples": 0}
        if self.proc is None:
            return out
        self.proc.terminate()
        try:
            self.proc.wait(timeout=5)
        except Exception:
            self.proc.kill()
        sm, mx, reasons = [], [], set()
        try:
            for ln in open(self.path):
                p = [x.strip() for x in ln.split(",")]
                if len(p) < 9:
                    continue
                try:
                    sm.append(float(p[1]))
                    mx.append(float(p[2]))
                except ValueError:
                    continue
                for name, v in zip(("hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"), p[5:9]):
                    if v.lower().startswith("active"):
                        reasons.add(name)
            os.unlink(self.path)
        except Exception:
            pass
        if sm:
            out.update(sm_mhz=float(np.median(sm)), sm_max_mhz=float(max(mx)), reasons=sorted(reasons), samples=len(sm))
        return out


def run_reorder():
    """--workload reorder: throughput of cuhpx_reorder (NESTED <-> RING, paper section III-B) on one
    GPU, one JSON line per case.  Device-timed with CUDA events (3 warm-ups, 20 calls); roofline HBM: algorithmic bytes =
    2 x batch x npix x element size (every element read once and written once)."""
    import torch

    from paper_2510_01785_b200 import binding as B

    peak, _ = load_peaks()
    for nside, batch, dt in [(1024, 8, torch.float32), (4096, 1, torch.float64), (4096, 4, torch.float32),
                             (2048, 8, torch.float64)]:
        npix = 12 * nside * nside
        a = torch.randn(batch, npix, dtype=dt, device="cuda")
        o = torch.empty_like(a)
        code = B._dtype_code(dt)
        for d, name in [(B.CUHPX_NEST2RING, "nest2ring"), (B.CUHPX_RING2NEST, "ring2nest")]:
            for _ in range(3):
                B.cuhpx_reorder(nside, batch, code, d, a, o)
            torch.cuda.synchronize()
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            e0.record()
            for _ in range(20):
                B.cuhpx_reorder(nside, batch, code, d, a, o)
            e1.record()
            torch.cuda.synchronize()
            ms = e0.elapsed_time(e1) / 20
            gbs = 2 * a.numel() * a.element_size() / ms / 1e6
            print(json.dumps({"op": name, "nside": nside, "batch": batch, "dtype": str(dt).split(".")[-1], "ms": ms,
                              "roofline": {"bound": "hbm", "achieved": gbs, "peak": peak, "unit": "GB/s", "frac": gbs / peak}}),
                  flush=True)


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=3)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--workload", default="cfg5", choices=sorted(synth.CONFIGS) + ["reorder"])
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--no-cpu-baseline", action="store_true")
    args = ap.parse_args()
    if args.workload == "reorder":
        run_reorder()
        return
    cfg = dict(synth.CONFIGS[args.workload])
    cfg["index"] = int(args.workload[3:]) - 1
    if args.impl == "reference":
        run_reference(args, cfg)
        return
    if args.gpus > 1 and "WORLD_SIZE" not in os.environ:
        # launched plainly: become the launcher of N ranks (one per GPU) of this same command line
        raise SystemExit(replicas.spawn_ranks(args.gpus, [os.path.abspath(__file__)] + sys.argv[1:]))

    import torch
    import torch.distributed as dist

    from paper_2510_01785_b200 import binding as B

    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device: the cuHPX path has no CPU fallback")
    torch.cuda.set_device(local)
    dev = torch.device("cuda", local)
    if world > 1:
        dist.init_process_group("nccl", device_id=dev)

    nside, lmax, mmax, batch = cfg["nside"], cfg["lmax"], cfg["mmax"], cfg["batch"]
    dt = cfg["dtype"]
    rdt = torch.float64 if dt == "f64" else torch.float32
    cdt = torch.complex128 if dt == "f64" else torch.complex64
    rbytes = 8 if dt == "f64" else 4
    npix, nalm = synth.npix(nside), synth.alm_count(lmax, mmax)

    # ---- inputs (synthetic, seeded): alm ~ (l+1)^-2 power law; the map inputs of the
    # analysis-type calls are the synthesised map (+ sigma = 0.01 pixel noise for cfg4), resident in HBM.
    t_inputs = time.perf_counter()
    alm_np = synth.powerlaw_alm(replicas.rank_seed(cfg["seed"], rank), lmax, mmax, batch)
    h_alm = torch.from_numpy(alm_np).to(cdt).pin_memory()
    t_inputs = time.perf_counter() - t_inputs
    torch.zeros(1, device=dev)
    torch.cuda.synchronize()  # context is up: what follows is the library's own first call
    T = B.Transform(nside, lmax, mmax, batch, rdt, dev)  # T.init_seconds: cuhpx_workspace_init alone
    stats = B.cuhpx_plan_stats(T.params)
    d_alm = h_alm.to(dev, non_blocking=True)
    d_map = T.alm2map(d_alm)
    if args.workload == "cfg4":
        d_map += 0.01 * torch.from_numpy(synth.gaussian_map(cfg["seed"] + 1, nside, batch)).to(rdt).to(dev)
    if args.workload in ("cfg1", "cfg3"):
        d_map = torch.from_numpy(synth.gaussian_map(cfg["seed"], nside, batch)).to(rdt).to(dev)
    h_map = d_map.cpu().pin_memory()
    d_alm_out = torch.empty_like(d_alm)
    d_map_out = torch.empty_like(d_map)
    h_alm_out = torch.empty_like(h_alm).pin_memory()
    h_map_out = torch.empty_like(h_map).pin_memory()
    torch.cuda.synchronize()

    ws = T.workspace
    P = T.params
    stages = ["fft_analysis", "legendre_analysis", "legendre_synthesis", "fft_synthesis"]

    def step():
        """One pass of the hot path: the four public C-ABI calls on resident buffers."""
        B.cuhpx_map2alm(*P, d_map, d_alm_out, None, ws)
        B.cuhpx_alm2map(*P, d_alm, d_map_out, ws)
        B.cuhpx_alm2map_adjoint(*P, d_map, d_alm_out, ws)
        B.cuhpx_map2alm_adjoint(*P, d_alm, d_map_out, None, ws)

    def staged_step(ev):
        """The same work through the stage-level entry points (the public calls are exactly these pairs), one
        CUDA-event pair per stage: the instrumented pass behind `roofline`, NOT the timed region of `value`."""
        def timed(name, fn):
            a = torch.cuda.Event(enable_timing=True)
            b = torch.cuda.Event(enable_timing=True)
            a.record()
            fn()
            b.record()
            ev.append((name, a, b))
        timed("fft_analysis", lambda: B.cuhpx_analysis_fft_stage(P, d_map, None, 1, ws))
        timed("legendre_analysis", lambda: B.cuhpx_analysis_legendre_stage(P, d_alm_out, 0, ws))
        timed("legendre_synthesis", lambda: B.cuhpx_synthesis_legendre_stage(P, d_alm, 0, ws))
        timed("fft_synthesis", lambda: B.cuhpx_synthesis_fft_stage(P, d_map_out, None, 0, ws))
        timed("fft_analysis", lambda: B.cuhpx_analysis_fft_stage(P, d_map, None, 0, ws))
        timed("legendre_analysis", lambda: B.cuhpx_analysis_legendre_stage(P, d_alm_out, 1, ws))
        timed("legendre_synthesis", lambda: B.cuhpx_synthesis_legendre_stage(P, d_alm, 1, ws))
        timed("fft_synthesis", lambda: B.cuhpx_synthesis_fft_stage(P, d_map_out, None, 1, ws))

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    # the sampler starts before the warm-up so that short workloads (a step of < 1 ms) still get samples under load
    sampler = ClockSampler(local)
    sampler.start()
    for _ in range(max(args.warmup, 3)):
        step()
    barrier()
    e0 = torch.cuda.Event(enable_timing=True)
    e1 = torch.cuda.Event(enable_timing=True)
    barrier()
    e0.record()
    for _ in range(args.steps):
        step()
    e1.record()
    barrier()
    # per-stage times: a separate instrumented pass of the same length
    ev = []
    for _ in range(args.steps):
        staged_step(ev)
    barrier()
    # a timed region shorter than the sampler's 100 ms period (cfg1-3) yields no sample: keep the same load running,
    # untimed, until nvidia-smi has reported a few
    t_extra = time.perf_counter()
    while sampler.count() < 3 and time.perf_counter() - t_extra < 2.0:
        for _ in range(50):
            step()
        torch.cuda.synchronize()
    clocks = sampler.stop()
    transforms_per_step = 4 * batch
    # whole job: every rank's transforms over the slowest rank's device time (no data-path collective)
    ms, units = replicas.reduce_timing(e0.elapsed_time(e1), transforms_per_step * args.steps, dev)
    value = units / (ms * 1e-3)

    stage_ms = {s: [] for s in stages}
    for name, a, b in ev:
        stage_ms[name].append(a.elapsed_time(b))
    stage_avg = {s: float(np.mean(v)) for s, v in stage_ms.items()}

    # ---- end to end through the public API with pinned host buffers: every step copies the four operators' inputs
    # host -> device and their results device -> host.  Copies run on their own streams and overlap the transforms
    # (three CUDA streams + events; each operator has its own device buffers so nothing is overwritten in flight).
    s_in, s_out = torch.cuda.Stream(dev), torch.cuda.Stream(dev)
    s_cmp = torch.cuda.current_stream(dev)
    d_in = [torch.empty_like(d_alm), torch.empty_like(d_map), torch.empty_like(d_map), torch.empty_like(d_alm)]
    d_out = [torch.empty_like(d_map), torch.empty_like(d_alm), torch.empty_like(d_alm), torch.empty_like(d_map)]
    h_in = [h_alm, h_map, h_map, h_alm]
    h_out = [h_map_out, h_alm_out, torch.empty_like(h_alm_out).pin_memory(), torch.empty_like(h_map_out).pin_memory()]
    ops = [T.alm2map, T.map2alm, T.alm2map_adjoint, T.map2alm_adjoint]
    ev_free_in = [None] * 4   # compute of the previous step has consumed d_in[k]
    ev_free_out = [None] * 4  # the previous step's copy-out of d_out[k] is done

    def e2e_step():
        ev_in, ev_done = [], []
        with torch.cuda.stream(s_in):
            for k in range(4):
                if ev_free_in[k] is not None:
                    s_in.wait_event(ev_free_in[k])
                d_in[k].copy_(h_in[k], non_blocking=True)
                e = torch.cuda.Event()
                e.record(s_in)
                ev_in.append(e)
        for k in range(4):
            s_cmp.wait_event(ev_in[k])
            if ev_free_out[k] is not None:
                s_cmp.wait_event(ev_free_out[k])
            ops[k](d_in[k], out=d_out[k])
            e = torch.cuda.Event()
            e.record(s_cmp)
            ev_done.append(e)
            ev_free_in[k] = e
        with torch.cuda.stream(s_out):
            for k in range(4):
                s_out.wait_event(ev_done[k])
                h_out[k].copy_(d_out[k], non_blocking=True)
                e = torch.cuda.Event()
                e.record(s_out)
                ev_free_out[k] = e

    def e2e_join():
        s_cmp.wait_stream(s_in)
        s_cmp.wait_stream(s_out)

    e2e_step()
    e2e_join()
    barrier()
    k_e2e = max(1, min(args.steps, 3))
    a = torch.cuda.Event(enable_timing=True)
    b = torch.cuda.Event(enable_timing=True)
    a.record()
    for _ in range(k_e2e):
        e2e_step()
    e2e_join()  # the timed region ends when the last result has landed in host memory
    b.record()
    barrier()
    ms_e2e, units_e2e = replicas.reduce_timing(a.elapsed_time(b), transforms_per_step * k_e2e, dev)
    e2e_value = units_e2e / (ms_e2e * 1e-3)
    map_bytes, alm_bytes = batch * npix * rbytes, batch * nalm * 2 * rbytes
    h2d = 2 * map_bytes + 2 * alm_bytes
    d2h = 2 * map_bytes + 2 * alm_bytes

    # ---- roofline of the dominant kernel + the other stages.  Legendre stages: flops of the
    # terms the kernels EXECUTE (insignificant (m, ring) pairs are skipped, R7) over the nominal FMA peak;
    # the SURVEY 8(d) all-terms figure T (4 + 4B) and the fraction of the FMA rate probed in this run are beside it.
    hbm_gbs, peak_src = load_peaks()
    terms_full, terms_exec = stats["legendre_terms_full"], stats["legendre_terms_executed"]
    # steps of terms_exec that the fp64 kernels no longer walk (late-start tables): not counted as work
    skipped = dict(zip(("legendre_analysis", "legendre_synthesis"), B.cuhpx_late_start_stats(T.params, T.workspace)))
    leg_flops_full = terms_full * (4 + 4 * batch)   # T (4 + 4B), T = nalm * 2 nside
    fft_bytes = batch * npix * rbytes + batch * stats["spectra_entries"] * 2 * rbytes  # map once + spectra once
    fma_ms, fma_cnt = B.cuhpx_fma_peak_probe(B.CUHPX_F64 if dt == "f64" else B.CUHPX_F32, 20000)
    fma_tflops = 2 * fma_cnt / (fma_ms * 1e-3) / 1e12
    traffic = {}
    tpath = os.path.join(ROOT, "profiles", "dram_traffic.json")
    if os.path.exists(tpath):
        try:
            traffic = json.load(open(tpath)).get(args.workload, {})
        except Exception:
            traffic = {}
    per_stage = {}
    for s in stages:
        if s.startswith("legendre"):
            ach = (terms_exec - skipped[s]) * (4 + 4 * batch) / (stage_avg[s] * 1e-3) / 1e12
            full = leg_flops_full / (stage_avg[s] * 1e-3) / 1e12
            per_stage[s] = {"bound": "alu", "achieved": ach, "peak": PEAK_TFLOPS[dt], "unit": "TFLOP/s",
                            "frac": ach / PEAK_TFLOPS[dt], "ms": stage_avg[s], "traffic": traffic.get(s),
                            "flops_counted": "walked terms x (4 + 4 B)", "terms_walked_frac": (terms_exec - skipped[s]) / terms_full,
                            "frac_of_fma_probe": ach / fma_tflops,
                            "algorithmic_all_terms": {"achieved": full, "frac": full / PEAK_TFLOPS[dt]}}
        else:
            ach = fft_bytes / (stage_avg[s] * 1e-3) / 1e9
            per_stage[s] = {"bound": "hbm", "achieved": ach, "peak": hbm_gbs, "unit": "GB/s", "frac": ach / hbm_gbs,
                            "ms": stage_avg[s], "traffic": traffic.get(s)}
    dominant = max(stages, key=lambda s: stage_avg[s])
    roofline = dict(per_stage[dominant])
    roofline.update(kernel=dominant, peak_source=("B200 nominal: 148 SM x 64/128 FMA lanes x 2 x 1.965 GHz"
                                                  if roofline["bound"] == "alu" else f"MEASURED_PEAKS.json ({peak_src})"),
                    fma_probe_tflops=fma_tflops, terms_executed_frac=(terms_exec - skipped.get(dominant, 0.0)) / terms_full,
                    timing="per-stage CUDA events of an instrumented pass over the stage-level calls, "
                           f"{args.steps} steps, separate from the timed region of `value`",
                    stages=per_stage)

    launches_per_step = int(4 * stats["fft_stage_launches"] + 2 * stats["legendre_analysis_launches"]
                            + 2 * stats["legendre_synthesis_launches"])

    # ---- CPU baseline: the oracle, as it stands, on a bounded sample (rank 0, N = 1 only)
    cpu = None
    if rank == 0 and world == 1 and not args.no_cpu_baseline:
        import oracle

        cores = oracle.num_threads()
        nr = max(8, (4 if nside >= 4096 else 16) * cores) if nside >= 1024 else 4 * nside - 1
        rings = oracle_sample_rings(nside, nr)
        frac = oracle_cost_fraction(nside, lmax, mmax, rings)
        a_in = alm_np[0] if dt == "f64" else alm_np[0].astype(np.complex64).astype(np.complex128)
        t0 = time.perf_counter()
        ref = oracle.alm2map_rings(nside, lmax, mmax, a_in, rings)
        tc = time.perf_counter() - t0
        # and use it: the bench refuses to print a number for a wrong transform
        T.alm2map(h_alm.to(dev), out=d_map_out)
        got = d_map_out[0].cpu().numpy().astype(np.float64)
        pieces = []
        for r in rings:
            n, start = oracle.ring_geometry(nside, r)[:2]
            pieces.append(got[start:start + n])
        got = np.concatenate(pieces)
        err = float(np.abs(got - ref).max() / np.abs(ref).max()) if dt == "f64" else \
            float(np.linalg.norm(got - ref) / np.linalg.norm(ref))
        tol = 1e-11 if dt == "f64" else 2e-5
        if err > tol:
            raise SystemExit(f"parity check against the oracle failed inside bench.py: {err:.3e} > {tol}")
        cpu = {"value": frac / tc, "unit": UNIT, "cores": cores, "kind": "oracle",
               "sample": f"alm2map on {len(rings)} of {4 * nside - 1} rings = {frac:.3e} of one transform in {tc:.1f} s "
                         f"(share of the oracle's operation count); GPU result on those rings matches to {err:.2e}"}

    if rank == 0:
        line = {
            "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps,
            "warmup": max(args.warmup, 3), "ms_per_step": ms / args.steps, "higher_is_better": True, "scaling": "weak",
            "vs_baseline": None, "dtype": dt, "data": "synthetic",
            "config": {"workload": workload_name(cfg), "step": "cuhpx_map2alm + cuhpx_alm2map + cuhpx_alm2map_adjoint + "
                       "cuhpx_map2alm_adjoint (the four public C-ABI calls)",
                       "transforms_per_step": transforms_per_step, "pixels_per_s": value * npix,
                       "l2_policy": f"inputs larger than L2 ({(map_bytes + alm_bytes) / 1e6:.0f} MB per call vs 126 MB)"
                       if map_bytes + alm_bytes > 126e6 else "inputs fit in L2 (latency-bound configuration)",
                       "replicas": world, "tables_first_call_s": T.init_seconds, "input_synthesis_s": t_inputs},
            "clocks": clocks,
            "e2e": {"value": e2e_value, "unit": UNIT, "h2d_bytes_per_step": h2d, "d2h_bytes_per_step": d2h,
                    "ms_per_step": ms_e2e / k_e2e, "steps": k_e2e},
            "gpu_launches": launches_per_step * args.steps,
            "roofline": roofline,
            "cpu_baseline": cpu,
        }
        print(json.dumps(line), flush=True)
    if world > 1:
        dist.destroy_process_group()


if __name__ == "__main__":
    main()
