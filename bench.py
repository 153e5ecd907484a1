#!/usr/bin/env python
"""bench.py -- Matching Pursuit on B200: MP iterations/s and achieved HBM GB/s vs the measured peak.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--config cfg3] [--impl reference]

One "step" = one pass of the whole hot path over one synthetic problem: column
normalisation of the dictionary (a0) followed by one complete mp_recover solve (a1-a8: init, the device-resident
loop of fused correlate+argmax / update+norm / stop test, return of x~, r, n_iter).  The default workload is
BASELINE.json's metric configuration (configs[2] = "cfg3": N=4096, M=16384 fp32 Bernoulli dictionary, K=256).
The dictionary (256 MiB) is larger than L2 (126 MB), so every MP iteration streams it from HBM: no L2 flush is
needed between timed iterations (stated in config.l2).

Prints ONE JSON line (rank 0).  Multi-GPU (torchrun): the path does not shard ("replicas only"):
every rank solves its own problem of the same shape; value = iterations of all ranks / max-over-ranks time.
"""
from __future__ import annotations

import argparse
import json
import os
import subprocess
import sys
import threading
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

from paper_0809_1833_b200 import synth  # noqa: E402  (seeded inputs only; numpy)

METRIC = "mp_iterations_per_s"
UNIT = "iterations/s"


def load_peaks():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        try:
            d = json.load(open(p))
            return float(d["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs)"
        except Exception:
            pass
    return 6650.0, "fallback (B200_PROFILING.md 6.65 TB/s)"


def load_tf32_peak():
    """Dense TF32 tensor peak in TFLOP/s: the measured sustained bf16 cuBLAS figure (the batched kernel is timed inside
    a long step) x the guide's nominal tf32/bf16 ratio 1.1/2.25."""
    ratio = 1.1 / 2.25
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        try:
            d = json.load(open(p))
            return float(d["bf16_tflops_sustained"]) * ratio, "measured bf16_tflops_sustained x 1.1/2.25 (nominal tf32/bf16)"
        except Exception:
            pass
    return 1400.0 * ratio, "fallback (B200_PROFILING.md 1.4 PFLOP/s sustained bf16) x 1.1/2.25"


K1_SOURCES = ["paper_0809_1833_b200/csrc/mp_persistent_ldg.cu", "paper_0809_1833_b200/csrc/mp_common.cuh", "paper_0809_1833_b200/csrc/mp_internal.h"]


def capture_is_stale(capture_commit: str):
    """A capture of the dominant kernel is only quoted if no later commit touched the kernel's sources: the last commit that did must be
    the capture's commit or one of its ancestors.  Returns a reason string when stale, "" when fine or when this cannot be told (no .git
    on the bench box, git missing)."""
    if not capture_commit or not os.path.isdir(os.path.join(ROOT, ".git")):
        return ""
    try:
        last = subprocess.run(["git", "-C", ROOT, "log", "-1", "--format=%H", "--"] + K1_SOURCES, capture_output=True, text=True, timeout=20)
        if last.returncode or not last.stdout.strip():
            return ""
        anc = subprocess.run(["git", "-C", ROOT, "merge-base", "--is-ancestor", last.stdout.strip(), capture_commit], capture_output=True, timeout=20)
    except Exception:
        return ""
    if anc.returncode != 1:               # 0 = ancestor-or-equal: fine; anything but 1 = git could not tell (unknown commit, shallow history)
        return ""
    return "captured at %s, but %s touched the kernel's sources later: re-capture" % (capture_commit, last.stdout.strip()[:7])


def ncu_traffic(kernel_name: str):
    """DRAM bytes per MP iteration of the dominant kernel -- a CONSTANT read from the committed ncu summary
    profiles/dominant_kernel_traffic.txt (dram__bytes_read.sum + dram__bytes_write.sum of one `ncu --set full` capture, divided
    by the iterations of that launch), not something this run measures.  Returns (with_hints, without_hints, provenance) or
    (None, None, reason).  Fails loudly when the capture is of another kernel than the one this run launched."""
    p = os.path.join(ROOT, "profiles", "dominant_kernel_traffic.txt")
    try:
        kv = {}
        for line in open(p):
            if "=" in line and not line.lstrip().startswith("#"):
                k, _, v = line.partition("=")
                kv[k.strip()] = v.split("#")[0].strip()
    except OSError:
        return None, None, "profiles/dominant_kernel_traffic.txt not found"
    if kv.get("kernel", "") not in kernel_name:
        raise SystemExit("profiles/dominant_kernel_traffic.txt is a capture of '%s' but this run launched '%s': re-capture it"
                         % (kv.get("kernel"), kernel_name))
    stale = capture_is_stale(kv.get("commit", ""))
    if stale:
        return None, None, "profiles/dominant_kernel_traffic.txt not used: " + stale
    prov = ("constant from profiles/dominant_kernel_traffic.txt (ncu --set full, %s, commit %s), multiplied by this run's iterations"
            % (kv.get("capture", "?"), kv.get("commit", "?")))
    return float(kv["dram_bytes_per_iteration"].split()[0]), float(kv["dram_bytes_per_iteration_no_hints"].split()[0]), prov


class ClockSampler:
    """nvidia-smi clocks/throttle reasons DURING the timed region (B200_PROFILING.md clocks line)."""
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,"
         "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")

    def __init__(self, index: int):
        self.index, self.rows, self.proc = index, [], None

    def start(self):
        try:
            self.proc = subprocess.Popen(["nvidia-smi", "-i", str(self.index), f"--query-gpu={self.Q}",
                                          "--format=csv,noheader,nounits", "-lms", "100"],
                                         stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            threading.Thread(target=self._read, daemon=True).start()
        except Exception:
            self.proc = None

    def _read(self):
        for line in self.proc.stdout:
            self.rows.append([c.strip() for c in line.split(",")])

    def stop(self):
        if self.proc is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        time.sleep(0.15)
        self.proc.terminate()
        sm, mx, reasons = [], None, set()
        for r in self.rows:
            try:
                sm.append(float(r[0])); mx = float(r[1])
            except Exception:
                continue
            for name, v in zip(("hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"), r[3:7]):
                if v.lower().startswith("active"):
                    reasons.add(name)
        return {"sm_mhz": float(np.median(sm)) if sm else None, "sm_max_mhz": mx, "reasons": sorted(reasons), "samples": len(sm)}


def build_problem(cfg: synth.Config, seed: int):
    """Host-side seeded inputs.  Returns raw dictionary [M,N] fp32 and Y [B,N] fp32.
    y = Psi x is formed from the dictionary the solver will see; for Gaussian configs the columns are normalised
    on the DEVICE by the product kernel before encoding, so this returns (psi_raw, X, S) and the caller encodes."""
    psi_raw = synth.make_dictionary(cfg, seed)
    X = np.zeros((cfg.B, cfg.M)); S = np.zeros((cfg.B, cfg.K), dtype=np.int64)
    for b in range(cfg.B):
        X[b], S[b] = synth.sparse_signal(cfg.M, cfg.K, seed, cfg.values, signal=b)
    return psi_raw, X, S


def config_dict(cfg, world=1, **more):
    """The `config` object of a JSON line: the same keys on both arms (the driver compares them)."""
    N, M = cfg.N, cfg.M
    d = {"workload": workload_name(cfg),
         "step": "mp_normalize_columns + %s (whole solve to the eps stop)" % ("mp_recover" if cfg.B == 1 else "mp_recover_batched"),
         "l2": "dictionary 4NM = %.0f MiB > 126 MB L2: inputs larger than L2, no flush" % (4.0 * N * M / 2**20)
               if 4.0 * N * M > 126e6 else "dictionary fits in L2 (cache-resident regime, by design of this config)",
         "parallelism": "replicas only" if world > 1 else "1 GPU"}
    d.update(more)
    return d


def run_reference(args, cfg):
    """--impl reference: the CPU oracle, as it stands, on the box's host cores; each step = a bounded sample
    (max_iter capped) of the same workload."""
    import oracle
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    sys.path.insert(0, os.path.join(ROOT, "tests"))
    import problems
    pb = problems.make_problem(cfg, seed=1)
    threads = oracle.default_threads()
    y = pb.Y[0].astype(np.float64)
    t0 = time.perf_counter(); oracle.mp(pb.psi32, y, cfg.eps, 4, threads); per_it = (time.perf_counter() - t0) / 4
    budget = 150.0 / max(1, args.steps + args.warmup)
    T = int(max(4, min(cfg.max_iter, budget / per_it)))
    for _ in range(args.warmup):
        oracle.mp(pb.psi32, y, cfg.eps, T, threads)
    t0 = time.perf_counter(); its = 0; ran = 0
    for _ in range(args.steps):
        ran = oracle.mp(pb.psi32, y, cfg.eps, T, threads).n_iter
        its += ran
    dt = time.perf_counter() - t0
    v = its / dt
    sample = (f"first {ran} MP iterations of {cfg.name} per step (iteration cap {T}; {'the oracle stopped by eps' if ran < T else 'capped'}; "
              f"float64 C oracle, OpenMP over atoms, {threads} threads)")
    print(json.dumps({
        "impl": "reference", "metric": METRIC, "value": v, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
        "warmup": args.warmup, "ms_per_step": 1e3 * dt / args.steps, "higher_is_better": True, "scaling": "weak",
        "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": config_dict(cfg, args.gpus), "iterations_per_step": ran, "sample": sample,
        "cpu_baseline": {"value": v, "unit": UNIT, "cores": threads, "kind": "oracle", "sample": sample},
        "e2e": {"value": v, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0}))


def aggregate(dist, elapsed_local, units_local, device):
    """Whole-job figures of a replicas-only run: the elapsed time is the MAX over ranks, the
    units (MP iterations) are the SUM over ranks.  `dist` is torch.distributed or None (single process)."""
    import torch
    t = torch.tensor([float(elapsed_local)], dtype=torch.float64, device=device)
    u = torch.tensor([float(units_local)], dtype=torch.float64, device=device)
    if dist is not None and dist.is_initialized() and dist.get_world_size() > 1:
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
        dist.all_reduce(u, op=dist.ReduceOp.SUM)
    return float(t.item()), float(u.item())


def workload_name(cfg):
    return (f"{cfg.name}: {'single-signal' if cfg.B == 1 else 'batched'} MP fp32, N={cfg.N}, M={cfg.M}, K={cfg.K}, {cfg.dictionary} dictionary, "
            f"eps={cfg.eps:g}, max_iter={cfg.max_iter}" + (f", B={cfg.B}" if cfg.B > 1 else ""))


def cpu_baseline(cfg, psi32, y32):
    """The oracle as it stands on this box's host cores, bounded sample (about 10-20 s)."""
    import oracle
    threads = oracle.default_threads()
    y = y32.astype(np.float64)
    t0 = time.perf_counter(); oracle.mp(psi32, y, cfg.eps, 4, threads); per_it = (time.perf_counter() - t0) / 4
    T = int(max(4, min(cfg.max_iter, 12.0 / per_it)))
    t0 = time.perf_counter(); res = oracle.mp(psi32, y, cfg.eps, T, threads); dt = time.perf_counter() - t0
    return {"value": res.n_iter / dt, "unit": UNIT, "cores": threads, "kind": "oracle",
            "sample": f"first {res.n_iter} MP iterations of {cfg.name} (float64 C oracle, OpenMP over atoms, {threads} threads)"}


class Workload:
    """One configuration resident in HBM: seeded inputs, outputs and workspace."""

    def __init__(self, torch, mp, cfg, seed, dev):
        self.torch, self.mp, self.cfg, self.dev = torch, mp, cfg, dev
        self.psi_raw, self.X, self.S = build_problem(cfg, seed)
        self.psi_d = torch.from_numpy(self.psi_raw).to(dev)
        mp.mp_normalize_columns(self.psi_d)               # so y can be encoded from the bits the solver sees
        torch.cuda.synchronize()
        self.psi32 = self.psi_d.cpu().numpy() if cfg.dictionary == "gaussian" else self.psi_raw
        self.Y = np.stack([synth.encode(self.psi32, self.X[b], self.S[b]) for b in range(cfg.B)])
        self.y_d = torch.from_numpy(self.Y).to(dev)
        N, M, B = cfg.N, cfg.M, cfg.B
        self.ws = torch.empty(mp.mp_workspace_bytes(N, M, B) + 256, dtype=torch.uint8, device=dev)
        self.x_d = torch.empty(B, M, dtype=torch.float32, device=dev)
        self.r_d = torch.empty(B, N, dtype=torch.float32, device=dev)
        self.n_d = torch.empty(B, dtype=torch.int32, device=dev)

    def normalize(self):
        self.mp.mp_normalize_columns(self.psi_d)                                     # a0 (idempotent on unit columns)

    def solve(self):
        c = self.cfg
        if c.B == 1:
            self.mp.mp_recover(self.psi_d, self.y_d[0], c.eps, c.max_iter, x=self.x_d[0], r=self.r_d[0], n_iter=self.n_d, workspace=self.ws)
        else:
            self.mp.mp_recover_batched(self.psi_d, self.y_d, c.eps, c.max_iter, X=self.x_d, R=self.r_d, n_iter=self.n_d, workspace=self.ws)

    def timed(self, steps, warmup, gpu_index, dist=None):
        """W warm-up steps, then K steps timed with CUDA events on the launching stream (barrier + synchronise on both sides),
        nvidia-smi clocks sampled during the timed region.  One retry if the region saw a thermal / hardware slowdown."""
        torch, mp = self.torch, self.mp
        stream = torch.cuda.current_stream()
        for attempt in range(2):
            # the sampler runs from the warm-up on (the same load as the timed steps): a short timed region still gets samples
            clocks = ClockSampler(gpu_index); clocks.start()
            for _ in range(warmup):
                self.normalize(); self.solve()
            torch.cuda.synchronize()
            ev = [torch.cuda.Event(enable_timing=True) for _ in range(2 * steps + 2)]
            if dist: dist.barrier()
            torch.cuda.synchronize()
            l0 = mp.mp_launch_count()
            ev[0].record(stream)
            for k in range(steps):
                self.normalize()
                ev[2 + 2 * k].record(stream)
                self.solve()
                ev[3 + 2 * k].record(stream)
            ev[1].record(stream)
            torch.cuda.synchronize()
            if dist: dist.barrier()
            launches = mp.mp_launch_count() - l0
            clk = clocks.stop()
            bad = [r for r in clk.get("reasons", []) if r in ("hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown")]
            if not bad or dist:
                break
            clk["rejected_once"] = bad
        ms_solve = [ev[2 + 2 * k].elapsed_time(ev[3 + 2 * k]) for k in range(steps)]
        return {"ms_total": ev[0].elapsed_time(ev[1]), "solve_ms": float(np.mean(ms_solve)), "launches": int(launches), "clocks": clk,
                "its_per_step": int(self.n_d.sum().item()), "its_max": int(self.n_d.max().item())}


def probe_read_gbs(torch, mp, dev, nbytes, passes, reps=3):
    """GB/s of the library's read-only streaming diagnostic (mp_probe_read: the item loop of the single-signal kernel, no barrier,
    no argmax) over a buffer of `nbytes`: the L2 read rate when the buffer fits in L2, the HBM read rate when it is much larger.
    Outside every timed region of the metric; best of `reps` after one warm-up launch."""
    unit = 148 * 8192
    nbytes = max(unit, (int(nbytes) + unit - 1) // unit * unit)
    buf = torch.ones(nbytes // 4, dtype=torch.float32, device=dev)
    sink = torch.zeros(1, dtype=torch.float32, device=dev)
    stream = torch.cuda.current_stream()
    mp.mp_probe_read(buf, max(1, passes // 4), sink=sink)
    torch.cuda.synchronize()
    best, read = 0.0, 0
    for _ in range(reps):
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record(stream)
        read = mp.mp_probe_read(buf, passes, sink=sink)
        e1.record(stream)
        torch.cuda.synchronize()
        best = max(best, read / (e0.elapsed_time(e1) * 1e-3) / 1e9)
    del buf
    torch.cuda.empty_cache()
    return {"gbs": best, "buffer_bytes": nbytes, "passes": passes, "bytes_read_per_launch": read,
            "source": "mp_probe_read (read-only 128-bit streaming loop of the single-signal kernel, one CTA per SM), CUDA events, best of %d, this run" % reps}


def l2_plan_of(mp):
    """The L2 plan of the last register-streaming launch, as the library reports it."""
    return {"reversed_order_on_odd_iterations": bool(mp.mp_get_int("info_l2_pingpong")),
            "pinned_mb": int(mp.mp_get_int("info_l2_resident_mb")),
            "items_drawn_from_counter": bool(mp.mp_get_int("info_l2_dynamic")),
            "l2_bytes": int(mp.mp_get_int("info_l2_bytes"))}   # cudaDevAttrL2CacheSize: the plan's thresholds are fractions of it


L2_RESIDENT_MAX_BYTES = 100e6      # dictionaries up to here are served by the 126 MB L2 after the first iteration


def roofline_of(mp, cfg, m, traffic_per_it=None, traffic_src=None, l2_probe=None):
    """The roofline object of the dominant kernel for one measured workload."""
    N, M, B = cfg.N, cfg.M, cfg.B
    its_max, solve_ms = m["its_max"], m["solve_ms"]
    peak, peak_src = load_peaks()
    if B > 1 and mp.mp_get_int("info_tc_clusters"):
        # batched path: the contraction Psi^T R on the tensor cores.  Algorithmic flops per lock-step iteration =
        # 3 x 2NMB (three TF32 products per fp32-accurate product); the dictionary is L2-resident (64 MiB).
        tpeak, tsrc = load_tf32_peak()
        alg_flops = its_max * 3.0 * 2.0 * N * M * B
        ach = alg_flops / (solve_ms * 1e-3) / 1e12
        return {"bound": "tensor", "achieved": ach, "peak": tpeak, "unit": "TFLOP/s", "frac": ach / tpeak, "traffic": None,
                "peak_source": tsrc, "kernel": mp_kernel_name(mp), "algorithmic_flops_per_launch": alg_flops,
                "kernel_ms": solve_ms, "us_per_lockstep_iteration": 1e3 * solve_ms / max(its_max, 1),
                "lockstep_iterations": its_max}
    # algorithmic bytes per launch: each iteration streams the dictionary once (4NM) and re-reads the winning atom (4N)
    # (SURVEY.md 8(d)); the batched loop runs until its slowest signal stops.
    alg_bytes = its_max * (4.0 * N * M + 4.0 * N * B)
    achieved = alg_bytes / (solve_ms * 1e-3) / 1e9
    streaming = 4.0 * N * M > L2_RESIDENT_MAX_BYTES
    rl = {"bound": "hbm", "regime": "hbm-streaming" if streaming else "l2-resident",
          "achieved": achieved, "peak": peak, "unit": "GB/s", "frac": achieved / peak,
          "traffic": traffic_per_it * its_max if traffic_per_it else None, "traffic_source": traffic_src, "peak_source": peak_src,
          "kernel": mp_kernel_name(mp, B > 1), "algorithmic_bytes_per_launch": alg_bytes, "kernel_ms": solve_ms,
          "us_per_iteration": 1e3 * solve_ms / max(its_max, 1)}
    if not streaming and l2_probe:
        # cache-resident regime (north_star: "or L2 bandwidth when Psi fits in L2"): the roofline is the L2 read rate, measured in
        # this run by the library's read-only probe over a buffer of the dictionary's own size
        rl.update({"bound": "l2", "peak": l2_probe["gbs"], "frac": achieved / l2_probe["gbs"], "peak_source": l2_probe["source"],
                   "l2_probe": l2_probe, "frac_vs_hbm_peak": achieved / peak, "hbm_peak": peak})
    if traffic_per_it and streaming:
        rl["dram_achieved"] = traffic_per_it * its_max / (solve_ms * 1e-3) / 1e9
        rl["dram_frac"] = rl["dram_achieved"] / peak
    return rl


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=5)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--config", default="cfg3")
    ap.add_argument("--impl", default="b200", choices=["b200", "reference"])
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--no-extra", action="store_true", help="skip the no-hint leg, the read probe and the cfg1 / cfg2 / cfg4 sweep / cfg5 figures of the default run")
    ap.add_argument("--max-iter", type=int, default=None, help="override the config's iteration cap (profiling runs)")
    ap.add_argument("--f64", action="store_true", help="double-precision path (mp_recover_f64) on the same workload shape")
    ap.add_argument("--omp", action="store_true", help="Orthogonal MP (mp_recover_omp) on the same workload")
    ap.add_argument("--signs", action="store_true", help="sign-packed Bernoulli dictionary (mp_recover_signs); Bernoulli configs only")
    ap.add_argument("--phase", default=None, metavar="RHO,SIGMA[,TRIALS]",
                    help="one cell of the paper's Fig. 1 phase diagram (P:92-106): M=1000, N=rho*M, K=sigma*M, TRIALS independent "
                         "problems each with its own Bernoulli dictionary, eps=1e-7, T=N, solved by one mp_recover_many launch")
    ap.add_argument("--knob", action="append", default=[], metavar="NAME=VALUE", help="mp_set_int knob (profiling runs)")
    args = ap.parse_args()
    if args.config == "cfg4":
        # the size sweep of BASELINE.json configs[3]: one full bench line per dictionary size (4 MiB ... 1 GiB), each from a
        # fresh process so that no state carries over between sizes
        for m in (2048, 4096, 8192, 16384, 32768):
            argv = [a if a != "cfg4" else "cfg4_%d" % m for a in sys.argv[1:]]
            subprocess.run([sys.executable, os.path.abspath(__file__)] + argv, check=True)
        return
    cfg = synth.config(args.config)
    if args.max_iter is not None:
        cfg = synth.Config(**{**cfg.__dict__, "max_iter": args.max_iter})
    if args.impl == "reference":
        return run_reference(args, cfg)
    if args.warmup < 3:
        print("note: warmup < 3 breaks the timing rules; use only for profiling runs", file=sys.stderr)

    import torch
    import paper_0809_1833_b200 as mp   # raises if the CUDA library is missing: there is no fallback

    for kv in args.knob:
        name, _, val = kv.partition("=")
        mp.mp_set_int(name, int(val))
    if args.phase:
        return run_phase(args, torch, mp)
    if args.f64:
        return run_f64(args, cfg, torch, mp)
    if args.omp:
        return run_omp(args, cfg, torch, mp)
    if args.signs:
        return run_signs(args, cfg, torch, mp)
    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device (no CPU fallback)")
    torch.cuda.set_device(local)
    dist = None
    if world > 1:
        import torch.distributed as dist
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))
    dev = torch.device("cuda", local)

    # ---- inputs: seeded, synthetic, resident in HBM before the timed region; K steps timed on the device ---------------
    wl = Workload(torch, mp, cfg, 1 + rank, dev)
    N, M, B = cfg.N, cfg.M, cfg.B
    m = wl.timed(args.steps, args.warmup, local, dist)
    ms_total_max, its_sum = aggregate(dist, m["ms_total"], float(m["its_per_step"] * args.steps), dev)
    value = its_sum / (ms_total_max * 1e-3)

    # ---- roofline of the dominant kernel (the persistent MP loop; one launch per solve) -------------------------
    per_it = per_it_off = tsrc = None
    if args.config == "cfg3" and not args.knob and args.max_iter is None and mp.mp_get_int("info_algo") == 3:
        per_it, per_it_off, tsrc = ncu_traffic(mp_kernel_name(mp, False))
    l2p = None
    if B == 1 and world == 1 and 4.0 * N * M <= L2_RESIDENT_MAX_BYTES:          # cache-resident config: roofline = the L2 read rate (probe over 64 MiB)
        l2p = probe_read_gbs(torch, mp, dev, 64 << 20, passes=400)
    roofline = roofline_of(mp, cfg, m, per_it, tsrc, l2_probe=l2p)
    if mp.mp_get_int("info_algo") == 3:
        roofline["l2_plan"] = l2_plan_of(mp)
    if per_it and "dram_frac" in roofline:
        # frac can exceed 1: ~88 MB of the dictionary are pinned in L2 (L2::evict_last loads) and odd iterations visit the rows in
        # reverse order, so that the rows read last are read first again: the kernel moves fewer HBM bytes per iteration than 4NM.
        roofline["note"] = ("frac = algorithmic bytes (4NM per iteration) / time against the HBM peak; it exceeds 1 because part of the "
                            "dictionary is served by L2 every iteration (88 MB of rows pinned by evict_last loads + the rows read last "
                            "in one iteration are read first in the next): ncu DRAM traffic is %.1f MB per iteration against "
                            "%.1f MB algorithmic (profiles/launches_r02.md); dram_frac is that traffic against the same peak; "
                            "no_hint is the same launch with both switched off (every byte from HBM), timed in this run"
                            % (per_it / 1e6, (4.0 * N * M + 4.0 * N) / 1e6))
    if B > 1 and roofline["bound"] == "tensor":
        roofline["note"] = "see profiles/batched_r02.md for what limits the contraction and the per-iteration chain"

    # ---- the same launch with the L2 residency hints OFF (every dictionary byte from HBM): outside the headline's timed region ----
    extra = None
    default_run = args.config == "cfg3" and not args.knob and args.max_iter is None and world == 1 and not args.no_extra
    if default_run:
        mp.mp_set_int("l2_resident_mb", 1); mp.mp_set_int("pingpong", 1)
        try:
            mo = wl.timed(3, 3, local)
        finally:
            mp.mp_set_int("l2_resident_mb", 0); mp.mp_set_int("pingpong", 0)
        ro = roofline_of(mp, cfg, mo, per_it_off, tsrc)
        roofline["no_hint"] = {"us_per_iteration": ro["us_per_iteration"], "achieved": ro["achieved"], "frac": ro["frac"],
                               "dram_frac": ro.get("dram_frac"), "steps": 3, "warmup": 3, "clocks": mo["clocks"],
                               "knob": "l2_resident_mb=1 pingpong=1 (no pinned rows, same visiting order every iteration): all 4NM bytes per iteration come from HBM"}

    if default_run:
        # the same-run anchor of the 1.02 / 1.47: what a read-only stream of the kernel's own access pattern gets from HBM (1 GiB buffer)
        hb = probe_read_gbs(torch, mp, dev, 1 << 30, passes=8)
        roofline["read_ceiling_hbm"] = {**hb, "frac_of_copy_peak": hb["gbs"] / roofline["peak"]}

    # ---- e2e: the host-buffer C-ABI call, H2D of the dictionary and y and D2H of x, r, n_iter inside the timed region ----
    e2e = None
    if not args.no_e2e:
        e2e = e2e_leg(args, torch, mp, cfg, wl, dist, local, dev)

    cb = None
    if rank == 0 and not args.no_cpu_baseline and world == 1:
        cb = cpu_baseline(cfg, wl.psi32, wl.Y[0])

    # ---- the other regimes DESIGN.md quotes, measured in this same run (own warm-up, own clocks sample; not part of `value`) ----
    if default_run:
        del wl
        torch.cuda.empty_cache()
        extra = {}
        # the L2 read rate of this box, once, for every cache-resident leg: the probe over 64 MiB (cfg2's size; north_star: "L2 bandwidth
        # when Psi fits in L2").  Smaller buffers would under-fill the probe's own grid (8 KiB items, 148 x 16 warps), not the L2.
        l2p64 = probe_read_gbs(torch, mp, dev, 64 << 20, passes=400)
        roofline["read_ceiling_l2"] = l2p64
        # the whole size sweep of BASELINE.json configs[3] (4 MiB ... 1 GiB, across the L2-to-HBM transition), cfg1, cfg2 and cfg5
        for name in ("cfg1", "cfg2", "cfg4_2048", "cfg4_4096", "cfg4_8192", "cfg4_16384", "cfg4_32768", "cfg5"):
            small = name in ("cfg1", "cfg4_2048", "cfg4_4096", "cfg4_16384")
            extra[name] = extra_leg(torch, mp, synth.config(name), local, dev, steps=3 if small else 5, l2_probe=l2p64)

    if rank == 0:
        print(json.dumps({
            "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": args.warmup,
            "ms_per_step": ms_total_max / args.steps, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
            "dtype": "f32", "data": "synthetic",
            "config": config_dict(cfg, world), "iterations_per_step": m["its_per_step"],
            "time_to_recovery_ms": m["solve_ms"], "gpu_launches": m["launches"], "clocks": m["clocks"],
            "roofline": roofline, "cpu_baseline": cb, "e2e": e2e, "extra": extra}))
    if dist:
        dist.destroy_process_group()


def extra_leg(torch, mp, cfg, local, dev, steps=5, warmup=3, l2_probe=None):
    """One of the other regimes (cfg1, cfg2, the cfg4 sizes: L2-resident up to 64 MiB, 1 GiB from HBM; cfg5: batched tensor-core),
    same protocol as the headline: W warm-ups, K timed steps, CUDA events, nvidia-smi clocks during its own timed region (one retry
    if that region saw a slowdown flag).  L2-resident sizes are stated against the L2 read rate of the probe (roofline.read_ceiling_l2)."""
    wl = Workload(torch, mp, cfg, 1, dev)
    m = wl.timed(steps, warmup, local)
    algo = int(mp.mp_get_int("info_algo")) if cfg.B == 1 else None
    plan = l2_plan_of(mp) if algo == 3 else None
    probe = l2_probe if cfg.B == 1 and 4.0 * cfg.N * cfg.M <= L2_RESIDENT_MAX_BYTES else None
    rl = roofline_of(mp, cfg, m, l2_probe=probe)
    out = {"workload": workload_name(cfg), "bound": rl["bound"], "frac": rl["frac"], "achieved": rl["achieved"], "peak": rl["peak"],
           "unit": rl["unit"], "peak_source": rl["peak_source"], "kernel": rl["kernel"], "iterations_per_step": m["its_per_step"],
           "steps": steps, "warmup": warmup, "ms_per_solve": m["solve_ms"], "clocks": m["clocks"],
           "us_per_iteration": rl.get("us_per_iteration", rl.get("us_per_lockstep_iteration"))}
    for k in ("regime", "frac_vs_hbm_peak", "l2_probe"):
        if k in rl:
            out[k] = rl[k]
    if plan is not None:
        out["l2_plan"] = plan
    if rl["bound"] == "hbm" and rl["frac"] > 1.0:
        out["note"] = ("frac counts the algorithmic 4NM bytes per iteration against the HBM copy peak; it exceeds 1 because part of the dictionary "
                       "is served by L2 every iteration (l2_plan: pinned rows and/or reversed order on odd iterations), as in the headline "
                       "(roofline.note, roofline.dram_frac, roofline.no_hint); a read-only stream alone reaches roofline.read_ceiling_hbm")
    if algo is not None:
        out["algo"] = algo
        if algo == 4:
            out["note"] = ("one 16-CTA cluster holds the dictionary in shared memory for the whole solve (no L2 traffic for Psi after "
                           "the first pass): the iteration is bound by the exchange inside the cluster, frac is bytes/time against the L2 rate for scale")
    if cfg.B > 1:
        out["signal_iterations_per_s"] = m["its_per_step"] / (m["solve_ms"] * 1e-3)
    del wl
    torch.cuda.empty_cache()
    return out


def e2e_leg(args, torch, mp, cfg, wl, dist, local, dev):
    """The same metric through the HOST-buffer C-ABI calls.  Two figures ("the host to device dictionary transfer only
    takes place once, since all signals are encoded/decoded with the same dictionary"):
      per call     -- mp_recover_host: allocate + H2D(Psi, y) + normalise + solve + D2H(x, r, n_iter) + free, every step
      steady state -- the dictionary lives in a handle (mp_dictionary_create: H2D + normalise, once, outside the timed region);
                      per step only y goes up and x, r, n_iter come back (mp_recover_host_h / mp_recover_batched_host_h)
    `value` is the PER-CALL figure, the definition of round 1 (every input of the step, the dictionary included, crosses the bus
    inside the timed region), so that rounds compare like with like; the handle path is reported under `steady_state`."""
    N, M, B = cfg.N, cfg.M, cfg.B
    hp = torch.from_numpy(wl.psi_raw).pin_memory()
    hY = torch.from_numpy(wl.Y).pin_memory()
    single = B == 1

    def first():
        if single:
            return int(mp.mp_recover_host(hp, hY[0], cfg.eps, cfg.max_iter, normalize=True, device=local).n_iter.item())
        return int(mp.mp_recover_batched_host(hp, hY, cfg.eps, cfg.max_iter, normalize=True, device=local).n_iter.sum().item())

    for _ in range(2):
        first()
    if dist: dist.barrier()
    t0 = time.perf_counter(); its = 0
    for _ in range(args.steps):
        its += first()
    dt = time.perf_counter() - t0
    dt_max, its_e = aggregate(dist, dt, float(its), dev)
    per_call = {"value": its_e / dt_max, "unit": UNIT, "ms_per_step": 1e3 * dt_max / args.steps,
                "h2d_bytes_per_step": 4 * N * M + 4 * N * B, "d2h_bytes_per_step": 4 * M * B + 4 * N * B + 4 * B,
                "definition": "per call: the dictionary and y are uploaded from pinned host memory inside the timed region of every step "
                              "(round 1's definition; round 2 reported the handle path here, now under steady_state)",
                "note": "mp_recover%s_host: stream-ordered device allocations + H2D(Psi, y) + normalise + solve + D2H(x, r, n_iter) + free per step"
                        % ("" if single else "_batched")}

    with torch.cuda.device(local):
        h = mp.mp_dictionary_create(hp, normalize=True)

    def steady():
        if single:
            return int(mp.mp_recover_host_h(h, hY[0], cfg.eps, cfg.max_iter).n_iter.item())
        return int(mp.mp_recover_batched_host_h(h, hY, cfg.eps, cfg.max_iter).n_iter.sum().item())

    for _ in range(2):
        steady()
    if dist: dist.barrier()
    t0 = time.perf_counter(); its = 0
    for _ in range(args.steps):
        its += steady()
    dt = time.perf_counter() - t0
    mp.mp_dictionary_destroy(h)
    dt_max, its_e = aggregate(dist, dt, float(its), dev)
    per_call["steady_state"] = {
        "value": its_e / dt_max, "unit": UNIT, "ms_per_step": 1e3 * dt_max / args.steps,
        "h2d_bytes_per_step": 4 * N * B, "d2h_bytes_per_step": 4 * M * B + 4 * N * B + 4 * B,
        "note": "dictionary resident in an mp_dictionary handle (uploaded and normalised once, P:165); per step "
                "H2D(y) + solve + D2H(x, r, n_iter) through mp_recover%s_host_h, pinned host buffers" % ("" if single else "_batched")}
    return per_call


def run_f64(args, cfg, torch, mp):
    """The double-precision path (NEXT 3) on the same workload shape, 1 GPU: normalise + solve in float64, HBM roofline
    with 8NM bytes per iteration.  Same JSON contract, dtype "f64"."""
    dev = torch.device("cuda", 0)
    torch.cuda.set_device(0)
    N, M = cfg.N, cfg.M
    psi_d = torch.from_numpy(synth.make_dictionary(cfg, 1)).to(dev).double()
    mp.mp_normalize_columns_f64(psi_d)
    x, sup = synth.sparse_signal(M, cfg.K, 1, cfg.values, signal=0)
    order = np.sort(sup)
    y_d = (torch.from_numpy(x[order]).to(dev)[:, None] * psi_d[torch.from_numpy(order).to(dev)]).sum(0)
    eps = float(np.float32(cfg.eps))
    ws = torch.empty(mp.binding.lib.mp_workspace_bytes_f64(N, M) + 256, dtype=torch.uint8, device=dev)
    stream = torch.cuda.current_stream()
    for _ in range(args.warmup):
        mp.mp_normalize_columns_f64(psi_d); res = mp.mp_recover_f64(psi_d, y_d, eps, cfg.max_iter, workspace=ws)
    clocks = ClockSampler(0); clocks.start()
    torch.cuda.synchronize()
    ev = [torch.cuda.Event(enable_timing=True) for _ in range(2 * args.steps + 2)]
    l0 = mp.mp_launch_count()
    ev[0].record(stream)
    for k in range(args.steps):
        mp.mp_normalize_columns_f64(psi_d)
        ev[2 + 2 * k].record(stream)
        res = mp.mp_recover_f64(psi_d, y_d, eps, cfg.max_iter, workspace=ws)
        ev[3 + 2 * k].record(stream)
    ev[1].record(stream)
    torch.cuda.synchronize()
    clk = clocks.stop()
    launches = mp.mp_launch_count() - l0
    its = int(res.n_iter.item())
    ms_total = ev[0].elapsed_time(ev[1])
    solve_ms = float(np.mean([ev[2 + 2 * k].elapsed_time(ev[3 + 2 * k]) for k in range(args.steps)]))
    peak, peak_src = load_peaks()
    alg_bytes = its * (8.0 * N * M + 8.0 * N)
    ach = alg_bytes / (solve_ms * 1e-3) / 1e9
    cb = None
    if not args.no_cpu_baseline:
        import oracle
        psi_h = psi_d.cpu().numpy(); y_h = y_d.cpu().numpy(); th = oracle.default_threads()
        t0 = time.perf_counter(); oracle.mp(psi_h, y_h, eps, 4, th); per_it = (time.perf_counter() - t0) / 4
        T = int(max(4, min(cfg.max_iter, 12.0 / per_it)))
        t0 = time.perf_counter(); r = oracle.mp(psi_h, y_h, eps, T, th); dt = time.perf_counter() - t0
        cb = {"value": r.n_iter / dt, "unit": UNIT, "cores": th, "kind": "oracle",
              "sample": f"first {r.n_iter} MP iterations of {cfg.name} in float64 (C oracle, OpenMP over atoms, {th} threads)"}
    print(json.dumps({
        "metric": METRIC, "value": its * args.steps / (ms_total * 1e-3), "unit": UNIT, "n_gpus": 1, "steps": args.steps,
        "warmup": args.warmup, "ms_per_step": ms_total / args.steps, "higher_is_better": True, "scaling": "weak",
        "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": {"workload": workload_name(cfg).replace("MP fp32", "MP fp64") + ", double precision (float64 dictionary, 8NM bytes per iteration)",
                   "iterations_per_step": its, "step": "mp_normalize_columns_f64 + mp_recover_f64 (whole solve to the eps stop)",
                   "l2": "dictionary 8NM = %.0f MiB" % (8.0 * N * M / 2**20), "parallelism": "1 GPU"},
        "time_to_recovery_ms": solve_ms, "gpu_launches": int(launches), "clocks": clk,
        "roofline": {"bound": "hbm", "achieved": ach, "peak": peak, "unit": "GB/s", "frac": ach / peak, "traffic": None,
                     "peak_source": peak_src, "kernel": "mp_persistent_f64_kernel", "algorithmic_bytes_per_launch": alg_bytes,
                     "kernel_ms": solve_ms, "us_per_iteration": 1e3 * solve_ms / max(its, 1)},
        "cpu_baseline": cb, "e2e": None}))


def run_omp(args, cfg, torch, mp):
    """Orthogonal MP (NEXT 2) on the same workload, 1 GPU.  One step = normalise + one whole mp_recover_omp solve; the
    correlation pass (4NM bytes per iteration) is the algorithmic traffic, the refit's 16tN bytes are L2-resident."""
    dev = torch.device("cuda", 0)
    torch.cuda.set_device(0)
    N, M = cfg.N, cfg.M
    psi_raw, X, S = build_problem(cfg, seed=1)
    psi_d = torch.from_numpy(psi_raw).to(dev)
    mp.mp_normalize_columns(psi_d)
    torch.cuda.synchronize()
    psi32 = psi_d.cpu().numpy() if cfg.dictionary == "gaussian" else psi_raw
    y32 = synth.encode(psi32, X[0], S[0])
    y_d = torch.from_numpy(y32).to(dev)
    T = min(cfg.max_iter, 2 * cfg.K)          # OMP takes one step per atom of the support; 2K is a generous cap
    ws = torch.empty(mp.binding.lib.mp_workspace_bytes_omp(N, M, T) + 256, dtype=torch.uint8, device=dev)
    stream = torch.cuda.current_stream()
    for _ in range(args.warmup):
        mp.mp_normalize_columns(psi_d); res = mp.mp_recover_omp(psi_d, y_d, cfg.eps, T, workspace=ws)
    clocks = ClockSampler(0); clocks.start()
    torch.cuda.synchronize()
    ev = [torch.cuda.Event(enable_timing=True) for _ in range(2 * args.steps + 2)]
    l0 = mp.mp_launch_count()
    ev[0].record(stream)
    for k in range(args.steps):
        mp.mp_normalize_columns(psi_d)
        ev[2 + 2 * k].record(stream)
        res = mp.mp_recover_omp(psi_d, y_d, cfg.eps, T, workspace=ws)
        ev[3 + 2 * k].record(stream)
    ev[1].record(stream)
    torch.cuda.synchronize()
    clk = clocks.stop()
    launches = mp.mp_launch_count() - l0
    its = int(res.n_iter.item())
    ms_total = ev[0].elapsed_time(ev[1])
    solve_ms = float(np.mean([ev[2 + 2 * k].elapsed_time(ev[3 + 2 * k]) for k in range(args.steps)]))
    peak, peak_src = load_peaks()
    alg_bytes = its * (4.0 * N * M + 4.0 * N)
    ach = alg_bytes / (solve_ms * 1e-3) / 1e9
    err = float(np.linalg.norm(res.x.cpu().numpy() - X[0]) / np.linalg.norm(X[0]))
    cb = None
    if not args.no_cpu_baseline:
        import oracle
        th = oracle.default_threads()
        Tc = min(T, 64)
        t0 = time.perf_counter(); r = oracle.omp(psi32, y32.astype(np.float64), cfg.eps, Tc, nthreads=th); dt = time.perf_counter() - t0
        cb = {"value": r.n_iter / dt, "unit": UNIT, "cores": th, "kind": "oracle",
              "sample": f"first {r.n_iter} OMP iterations of {cfg.name} (float64 C oracle, OpenMP correlation, {th} threads)"}
    print(json.dumps({
        "metric": METRIC, "value": its * args.steps / (ms_total * 1e-3), "unit": UNIT, "n_gpus": 1, "steps": args.steps,
        "warmup": args.warmup, "ms_per_step": ms_total / args.steps, "higher_is_better": True, "scaling": "weak",
        "vs_baseline": None, "dtype": "f32", "data": "synthetic",
        "config": {"workload": workload_name(cfg).replace(" MP ", " Orthogonal MP ") + f" (iteration cap {T})",
                   "iterations_per_step": its, "step": "mp_normalize_columns + mp_recover_omp (whole solve to the eps stop)",
                   "rel_error_vs_true_x": err, "parallelism": "1 GPU"},
        "time_to_recovery_ms": solve_ms, "gpu_launches": int(launches), "clocks": clk,
        "roofline": {"bound": "hbm", "achieved": ach, "peak": peak, "unit": "GB/s", "frac": ach / peak, "traffic": None,
                     "peak_source": peak_src,
                     "kernel": ("mp_omp_persistent_kernel (basis slices stationary in shared memory)" if mp.mp_get_int("info_omp_algo") == 1
                                else "stream loop: sl_correlate_argmax_kernel + omp_* refit kernels"),
                     "algorithmic_bytes_per_launch": alg_bytes, "kernel_ms": solve_ms,
                     "us_per_iteration": 1e3 * solve_ms / max(its, 1)},
        "cpu_baseline": cb, "e2e": None}))


def run_signs(args, cfg, torch, mp):
    """MP on the sign-packed Bernoulli dictionary (NEXT 4), 1 GPU.  One step = pack the signs + one whole solve.  The
    iteration is ALU-bound: N*M conditional adds; peak = SMs x 128 fp32 lanes x max SM clock (B200_PROFILING.md counts)."""
    if cfg.dictionary != "bernoulli":
        raise SystemExit("--signs needs a Bernoulli configuration (cfg3)")
    dev = torch.device("cuda", 0)
    torch.cuda.set_device(0)
    N, M = cfg.N, cfg.M
    psi_raw, X, S = build_problem(cfg, seed=1)
    psi_d = torch.from_numpy(psi_raw).to(dev)
    y_d = torch.from_numpy(synth.encode(psi_raw, X[0], S[0])).to(dev)
    ws = torch.empty(mp.mp_workspace_bytes(N, M, 1) + 256, dtype=torch.uint8, device=dev)
    stream = torch.cuda.current_stream()
    for _ in range(args.warmup):
        bits, scale, n_bad = mp.mp_pack_signs(psi_d); res = mp.mp_recover_signs(bits, N, scale, y_d, cfg.eps, cfg.max_iter, workspace=ws)
    assert n_bad == 0
    clocks = ClockSampler(0); clocks.start()
    torch.cuda.synchronize()
    ev = [torch.cuda.Event(enable_timing=True) for _ in range(2 * args.steps + 2)]
    l0 = mp.mp_launch_count()
    ev[0].record(stream)
    for k in range(args.steps):
        bits, scale, n_bad = mp.mp_pack_signs(psi_d)
        ev[2 + 2 * k].record(stream)
        res = mp.mp_recover_signs(bits, N, scale, y_d, cfg.eps, cfg.max_iter, workspace=ws)
        ev[3 + 2 * k].record(stream)
    ev[1].record(stream)
    torch.cuda.synchronize()
    clk = clocks.stop()
    launches = mp.mp_launch_count() - l0
    its = int(res.n_iter.item())
    ms_total = ev[0].elapsed_time(ev[1])
    solve_ms = float(np.mean([ev[2 + 2 * k].elapsed_time(ev[3 + 2 * k]) for k in range(args.steps)]))
    sm = torch.cuda.get_device_properties(0).multi_processor_count
    peak = sm * 128 * 1.965e9 / 1e12                       # T lane-ops/s
    ach = its * float(N) * M / (solve_ms * 1e-3) / 1e12
    print(json.dumps({
        "metric": METRIC, "value": its * args.steps / (ms_total * 1e-3), "unit": UNIT, "n_gpus": 1, "steps": args.steps,
        "warmup": args.warmup, "ms_per_step": ms_total / args.steps, "higher_is_better": True, "scaling": "weak",
        "vs_baseline": None, "dtype": "f32", "data": "synthetic",
        "config": {"workload": workload_name(cfg) + ", dictionary as 1 sign bit per entry (N*M/8 = %.0f MiB, stationary in shared memory)" % (N * M / 8 / 2**20),
                   "iterations_per_step": its, "step": "mp_pack_signs + mp_recover_signs (whole solve to the eps stop)", "parallelism": "1 GPU"},
        "time_to_recovery_ms": solve_ms, "gpu_launches": int(launches), "clocks": clk,
        "roofline": {"bound": "alu", "achieved": ach, "peak": peak, "unit": "T conditional adds/s", "frac": ach / peak, "traffic": None,
                     "peak_source": "%d SMs x 128 fp32 lanes x 1.965 GHz, one lane-op per dictionary entry (a test plus an add is two)" % sm,
                     "kernel": "mp_persistent_signs_kernel", "kernel_ms": solve_ms, "us_per_iteration": 1e3 * solve_ms / max(its, 1)},
        "cpu_baseline": None, "e2e": None}))


def run_phase(args, torch, mp):
    """One (sigma, rho) cell of the paper's Fig. 1 experiment (NEXT 4), 1 GPU: TRIALS independent problems, each with its own
    Bernoulli dictionary (Eq. 13) and K nonzeros from U[-1, 1], eps = 1e-7, T = N.  One step = one
    mp_recover_many launch over all trials.  The dictionaries in flight are L2-resident by plan, so the bound is L2 bandwidth."""
    parts = [float(v) for v in args.phase.split(",")]
    rho, sigma = parts[0], parts[1]
    P = int(parts[2]) if len(parts) > 2 else 400
    M = 1000
    N = max(4, int(round(rho * M / 4.0)) * 4)                  # ld % 4 == 0 at the boundary: N rounded to a multiple of 4
    K = max(1, int(round(sigma * M)))
    cfg = synth.Config("phase", N, M, K, "bernoulli", "uniform", 1e-7, N, 1)
    dev = torch.device("cuda", 0)
    torch.cuda.set_device(0)
    psi_h = torch.empty((P, M, N), dtype=torch.float32).pin_memory()
    Y_h = torch.empty((P, N), dtype=torch.float32).pin_memory()
    X_true = np.zeros((P, M))
    for q in range(P):
        d = synth.make_dictionary(cfg, 1000 + q)
        x, S = synth.sparse_signal(M, K, 1000 + q, cfg.values)
        psi_h[q] = torch.from_numpy(d); Y_h[q] = torch.from_numpy(synth.encode(d, x, S)); X_true[q] = x
    psi_d, Y_d = psi_h.to(dev), Y_h.to(dev)
    stream = torch.cuda.current_stream()
    res = None
    signs = bool(args.signs)

    def step(ws):
        if signs:                  # the same cell from one sign bit per entry: pack the stacked dictionaries, one CTA per problem
            bits, scale, n_bad = mp.mp_pack_signs(psi_d.view(P * M, N))
            assert n_bad == 0
            return mp.mp_recover_signs_many(bits.view(P, M, -1), N, scale, Y_d, cfg.eps, cfg.max_iter, workspace=ws)
        return mp.mp_recover_many(psi_d, Y_d, cfg.eps, cfg.max_iter, workspace=ws)

    for _ in range(max(args.warmup, 1)):
        res = step(res.workspace if res else None)
    clocks = ClockSampler(0); clocks.start()
    torch.cuda.synchronize()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    l0 = mp.mp_launch_count()
    e0.record(stream)
    for _ in range(args.steps):
        res = step(res.workspace)
    e1.record(stream)
    torch.cuda.synchronize()
    clk = clocks.stop()
    launches = mp.mp_launch_count() - l0
    ms = e0.elapsed_time(e1) / args.steps
    its = int(res.n_iter.sum().item())
    # Eq. 14 per trial by the library's own scoring kernel (mp_reconstruction_error), outside the timed region
    Xt_d = torch.from_numpy(X_true.astype(np.float32)).to(dev)
    err_d = torch.empty(P, dtype=torch.float64, device=dev)
    for q in range(P):
        mp.mp_reconstruction_error(res.x[q], Xt_d[q], out=err_d[q:q + 1])
    err = err_d.cpu().numpy()
    ach = its * 4.0 * N * M / (ms * 1e-3) / 1e9
    l2_peak = 17500.0
    out = {
        "metric": METRIC, "value": its / (ms * 1e-3), "unit": UNIT, "n_gpus": 1, "steps": args.steps, "warmup": args.warmup,
        "ms_per_step": ms, "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f32", "data": "synthetic",
        "config": {"workload": f"phase-diagram cell rho={N / M:g}, sigma={K / M:g}: {P} trials, M={M}, N={N}, K={K}, own Bernoulli dictionary per trial, "
                               f"U[-1,1] nonzeros, eps=1e-07, T=N", "iterations_per_step": its, "step": "one mp_recover_many launch over all trials",
                   "l2": "by plan the dictionaries of the clusters in flight fit in L2; all trials together (%.0f MB) do not" % (P * 4.0 * N * M / 1e6),
                   "parallelism": "1 GPU"},
        "solves_per_s": P / (ms * 1e-3), "mean_error_pct_eq14": float(np.mean(err)), "mean_iterations": its / P,
        "plan": {"threads": mp.mp_get_int("info_many_threads"), "cluster": mp.mp_get_int("info_many_cluster"),
                 "stationary": mp.mp_get_int("info_many_stat"), "clusters_in_flight": mp.mp_get_int("info_many_clusters")},
        "gpu_launches": int(launches), "clocks": clk,
        "roofline": {"bound": "l2", "achieved": ach, "peak": l2_peak, "unit": "GB/s", "frac": ach / l2_peak, "traffic": None,
                     "peak_source": "plain 128-bit loads of an L2-resident buffer on this pool's B200 (profiles/persistent_r01.md: 17-18 TB/s)",
                     "kernel": "mp_many_kernel", "kernel_ms": ms, "algorithmic_bytes_per_launch": its * 4.0 * N * M},
    }
    if signs:
        sm = torch.cuda.get_device_properties(0).multi_processor_count
        peak = sm * 128 * 1.965e9 / 1e12
        ops = its * float(N) * M / 4.0 / (ms * 1e-3) / 1e12                    # one table lookup + add per four entries
        out["config"]["workload"] += "; dictionaries as 1 sign bit per entry, one CTA per problem, bits stationary in shared memory"
        out["config"]["step"] = "mp_pack_signs of the stacked dictionaries + one mp_recover_signs_many launch over all trials"
        out["plan"] = None
        out["roofline"] = {"bound": "alu", "achieved": ops, "peak": peak, "unit": "T lookup-adds/s", "frac": ops / peak, "traffic": None,
                           "peak_source": "%d SMs x 128 fp32 lanes x 1.965 GHz; the lookup scheme needs one add per four dictionary entries "
                                          "(plus a shift, a mask and a shared-memory load)" % sm,
                           "kernel": "mp_many_signs_kernel", "kernel_ms": ms}
    if not args.no_cpu_baseline:
        import oracle                                      # the cpu_baseline leg: the only use of the oracle in this mode
        th = oracle.default_threads()
        t0 = time.perf_counter(); n_ref = 0; q = 0
        while q < P and time.perf_counter() - t0 < 10.0:
            n_ref += oracle.mp(psi_h[q].numpy(), Y_h[q].numpy().astype(np.float64), float(np.float32(cfg.eps)), cfg.max_iter, th).n_iter; q += 1
        dt = time.perf_counter() - t0
        out["cpu_baseline"] = {"value": n_ref / dt, "unit": UNIT, "cores": th, "kind": "oracle",
                               "sample": f"the first {q} trials of the cell, one after another (float64 C oracle, OpenMP over atoms, {th} threads)"}
    if not args.no_e2e and not signs:
        Xh = torch.empty((P, M), dtype=torch.float32).pin_memory(); nh = torch.empty(P, dtype=torch.int32).pin_memory()
        t_best = None
        for _ in range(2):
            torch.cuda.synchronize(); t0 = time.perf_counter()
            pd = psi_h.to(dev, non_blocking=True); yd = Y_h.to(dev, non_blocking=True)
            r2 = mp.mp_recover_many(pd, yd, cfg.eps, cfg.max_iter, workspace=res.workspace)
            Xh.copy_(r2.x, non_blocking=True); nh.copy_(r2.n_iter, non_blocking=True)
            torch.cuda.synchronize(); dt = time.perf_counter() - t0
            t_best = dt if t_best is None else min(t_best, dt)
        out["e2e"] = {"value": int(nh.sum().item()) / t_best, "unit": UNIT, "h2d_bytes_per_step": int(psi_h.numel() * 4 + Y_h.numel() * 4),
                      "d2h_bytes_per_step": int(Xh.numel() * 4 + nh.numel() * 4), "ms_per_step": t_best * 1e3,
                      "note": "pinned host dictionaries and measurements -> device, mp_recover_many, x~ and n_iter -> pinned host, per step"}
    print(json.dumps(out))


def mp_kernel_name(mp, batched=None):
    try:
        if mp.mp_get_int("info_tc_clusters") and batched is not False:
            return ("mp_batched_tc_kernel (%d clusters x 4 CTAs, %d atoms/tile, %d stages)"
                    % (mp.mp_get_int("info_tc_clusters"), mp.mp_get_int("info_tc_at"), mp.mp_get_int("info_tc_stages")))
        return {1: "mp_persistent_kernel (TMA-staged)", 2: "stream loop",
                3: "mp_persistent_ldg_kernel (register-streaming)",
                4: "mp_many_kernel (one cluster, dictionary stationary in shared memory)"}[mp.mp_get_int("info_algo")]
    except Exception:
        return "?"


if __name__ == "__main__":
    main()
