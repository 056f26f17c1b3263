#!/usr/bin/env python
"""bench.py -- one JSON line for the tdx hot path.

A step = one pass of the whole hot path over one synthetic field of the chosen BASELINE.json config:
    x sweep -> y sweep -> cyclic z sweep of (I - alpha delta2)   (tdx_adi_sweep, PPT or PDD, tuned P)
    + the nm = nz/2+1 spanwise-wavenumber Helmholtz y-solves      (tdx_helmholtz_wavenumber_solve)
metric  = Gpts/s per sweep: real grid values solved per second, averaged over the four sweeps of a step
          (points of a step = 3 nx ny nz + 2 nx ny nm).
Launch: python bench.py --gpus N --steps K --warmup W   (N > 1: under torch.distributed.run, one rank per GPU; the
path shards as independent fields, weak scaling, no data-path collective).
--impl reference times the CPU oracle (oracle/) on the host cores on a bounded sample of the same workload.
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

from paper_1812_01178_b200 import configs  # noqa: E402

METRIC = "Gpts/s per ADI sweep direction (fp64 PDD/PPT); achieved HBM GB/s vs peak"
UNIT = "Gpts/s"
BYTES_PER_POINT = 16.0          # 8 B read + 8 B written per real grid value per sweep

# partitions per line for the per-line-shift Helmholtz solve (kx2 != 0): at most 16 rows per partition
TUNED_P_LINE = {1: 4, 2: 16, 3: 32, 4: 32, 5: 24, 6: 16}

PDD_GATE = 1e-11                # DESIGN.md reading A9: north_star's 1e-10 PDD bar applies where the a-priori dropped bound <= 1e-11

NCU_TRAFFIC_FILE = os.path.join(ROOT, "profiles", "r2_ncu_traffic.csv")


def ncu_traffic(workload, launch):
    """roofline.traffic: dram__bytes_read.sum + dram__bytes_write.sum per launch of the committed `ncu --set full` capture
    (profiles/r2_ncu_traffic.csv; the command is in profiles/r2_ncu_traffic.md) for exactly this workload, kernel
    instantiation and launch shape (tdx_last_launch()).  A kernel or launch-shape change finds no row: (None, reason)."""
    if not os.path.exists(NCU_TRAFFIC_FILE):
        return None, "no committed capture (profiles/r2_ncu_traffic.csv missing)"
    import csv
    with open(NCU_TRAFFIC_FILE) as f:
        for row in csv.DictReader(r for r in f if not r.startswith("#")):
            if row["workload"] == workload and row["launch"] == launch:
                return float(row["dram_bytes_read"]) + float(row["dram_bytes_write"]), "profiles/r2_ncu_traffic.csv (ncu --set full, per launch)"
    return None, "no committed ncu capture for %s on %s" % (launch, workload)


# tuned partitions per line (x, y, z, helmholtz-y) per config, mode PPT (exact for every P)
TUNED_P = {1: (4, 4, 4, 4), 2: (16, 8, 8, 8), 3: (32, 8, 8, 8), 4: (128, 32, 8, 16), 5: (256, 12, 16, 12), 6: (384, 8, 24, 8)}


def pdd_partitions(grid, cfg, direction, P_ppt):
    """P for a PDD sweep, by rule (never by hand): the PPT-tuned P if PDD is inside its regime there (a-priori bound
    tdx_pdd_dropped_bound <= PDD_GATE, PAPER.md:L152 'n >> p'), else the largest smaller divisor of the line length whose
    bound passes.  Returns (P, bound)."""
    n = (cfg.nx, cfg.ny, cfg.nz)[direction]
    for P in [P_ppt] + [d for d in range(P_ppt - 1, 1, -1) if n % d == 0]:
        if n // P < 2:
            continue
        bound = grid.pdd_dropped_bound(direction, P, cfg.alpha)
        if bound <= PDD_GATE:
            return P, bound
    return 1, 0.0                                               # P = 1 is the plain Thomas recurrence


def parse():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=10)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="tdx", choices=["tdx", "reference"])
    ap.add_argument("--config", type=int, default=5, help="BASELINE.json config number 1..5; 6 = the paper's own 3072x256x768 grid")
    ap.add_argument("--mode", default="ppt", choices=["ppt", "pdd", "thomas"])
    ap.add_argument("--P", default="", help="override partitions: Px,Py,Pz,Ph")
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--no-cpu", action="store_true")
    ap.add_argument("--e2e-steps", type=int, default=2)
    ap.add_argument("--no-step3", action="store_true", help="skip the extra 3-component staggered ADI step figure")
    ap.add_argument("--no-slab", action="store_true", help="skip `slab_y_sweep`: the y sweep of ONE field cut into y-slabs over the ranks "
                    "(NCCL neighbour exchange / all-gather; SURVEY 8(f) N3; strong scaling).  Default at every N; at N = 1 it is the "
                    "compute part of one rank of a 4-rank job.")
    ap.add_argument("--slab", action="store_true", help=argparse.SUPPRESS)      # round-1 opt-in, now the default
    ap.add_argument("--psweep", default="", help="P sweep table (e.g. 8,16,32,64): per direction and mode, time, GB/s, PDD bound, "
                                                 "error of sampled lines vs the oracle; prints a markdown table, not the JSON line")
    ap.add_argument("--selftest-ranks", action="store_true",
                    help="CPU-only check of the N>1 host logic over gloo (used by tests/test_bench_ranks_gloo.py)")
    return ap.parse_args()


# ---- N > 1 host logic (one process per GPU; the path shards as independent fields, no data-path collective) ----------
def init_dist(world, backend, local_rank=0):
    """Process group for the barrier and the max-over-ranks reduction only. MASTER_ADDR/PORT, RANK, WORLD_SIZE from env."""
    if world <= 1:
        return None
    import datetime
    import torch
    import torch.distributed as dist
    # a collective that never completes (a dead peer) aborts after two minutes instead of hanging the bench
    if backend == "nccl":
        nccl_log_setup()
        dist.init_process_group("nccl", device_id=torch.device("cuda", local_rank), timeout=datetime.timedelta(seconds=120))
    else:
        dist.init_process_group(backend, timeout=datetime.timedelta(seconds=120))
    return dist


def nccl_log_setup():
    """NCCL's own INIT lines (communicator size, transport, NVLS) go to a file per process, so the N > 1 line can say which
    communicator it really ran on without polluting stdout (the JSON line).  Respects a caller's NCCL_DEBUG settings."""
    if "NCCL_DEBUG" in os.environ:
        return
    d = os.path.join(ROOT, "gpurun_out")
    try:
        os.makedirs(d, exist_ok=True)
    except OSError:
        return
    os.environ["NCCL_DEBUG"] = "INFO"
    os.environ["NCCL_DEBUG_SUBSYS"] = "INIT,GRAPH"
    os.environ["NCCL_DEBUG_FILE"] = os.path.join(d, "nccl_%h_%p.log")


def nccl_log_summary():
    """What this process's NCCL log says: communicator sizes seen, whether NVLS (in-switch reduction) was set up."""
    import re
    pat = os.environ.get("NCCL_DEBUG_FILE", "")
    if not pat:
        return None
    path = pat.replace("%h", __import__("socket").gethostname()).replace("%p", str(os.getpid()))
    try:
        text = open(path, errors="replace").read()
    except OSError:
        return {"log": path, "error": "not written"}
    return {"log": os.path.relpath(path, ROOT), "nranks_seen": sorted({int(v) for v in re.findall(r"nranks (\d+)", text)}),
            "nvls": "NVLS" in text, "p2p": "P2P" in text, "lines": text.count("\n")}


def max_over_ranks(value, dist, device="cpu"):
    """Every multi-GPU number is the MAX over ranks of a device-side time."""
    if dist is None:
        return float(value)
    import torch
    t = torch.tensor([float(value)], device=device, dtype=torch.float64)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def rank_seed(cfg, rank):
    """Rank r solves its own field: same shape and recipe, seed shifted (weak scaling)."""
    return cfg.seed + 1000 * rank


def whole_job_value(cfg, world, steps, total_ms):
    return world * step_points(cfg) * steps / (total_ms * 1e-3) / 1e9


def selftest_ranks(args, rank, world):
    dist = init_dist(world, "gloo")
    cfg = configs.get(1)
    seeds = [rank_seed(cfg, r) for r in range(world)]
    assert len(set(seeds)) == world and seeds[0] == cfg.seed
    fake_ms = 10.0 * (rank + 1)                                   # slowest rank = world-1
    mx = max_over_ranks(fake_ms, dist)
    assert mx == 10.0 * world, (mx, world)
    val = whole_job_value(cfg, world, 2, mx)
    if dist is not None:
        dist.barrier()
    if rank == 0:
        print(json.dumps({"selftest": "ok", "world": world, "max_ms": mx, "value": val, "seeds": seeds}))
    if dist is not None:
        dist.destroy_process_group()


def measured_peak():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        try:
            return float(json.load(open(p))["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs)"
        except Exception:
            pass
    return 6650.0, "fallback (B200_PROFILING.md 6.65 TB/s)"


class ClockSampler(threading.Thread):
    """nvidia-smi clocks / throttle reasons DURING the timed region."""
    Q = "clocks.sm,clocks.max.sm,clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown," \
        "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap"

    def __init__(self, index):
        super().__init__(daemon=True)
        self.index, self.stop_flag, self.rows = index, threading.Event(), []

    def run(self):
        try:
            proc = subprocess.Popen(["nvidia-smi", "-i", str(self.index), "--query-gpu=" + self.Q, "--format=csv,noheader,nounits", "-lms", "100"],
                                    stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
        except Exception:
            return
        while not self.stop_flag.is_set():
            line = proc.stdout.readline()
            if not line:
                break
            self.rows.append([x.strip() for x in line.split(",")])
        proc.terminate()

    def summary(self):
        sm = [float(r[0]) for r in self.rows if r and r[0].replace(".", "").isdigit()]
        mx = [float(r[1]) for r in self.rows if len(r) > 1 and r[1].replace(".", "").isdigit()]
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        reasons = [n for k, n in enumerate(names) if any(len(r) > 2 + k and r[2 + k].lower().startswith("active") for r in self.rows)]
        return {"sm_mhz": float(np.median(sm)) if sm else None, "sm_max_mhz": max(mx) if mx else None,
                "reasons": reasons, "samples": len(sm)}


def step_points(cfg):
    return 3 * cfg.npts + 2 * cfg.nx * cfg.ny * cfg.nm


def sample_shapes(cfg):
    """Bounded sample of the workload for the CPU oracle: same grid lines, fewer of them (about 10-30 s of CPU work)."""
    budget = 250_000_000                                       # real values per sweep
    kx = max(1, min(cfg.nz, budget // (cfg.nx * cfg.ny)))      # planes for the x and y sweeps
    jz = max(1, min(cfg.ny, budget // (cfg.nx * cfg.nz)))      # rows for the z sweep
    mh = max(1, min(cfg.nm, budget // (2 * cfg.nx * cfg.ny)))  # wavenumbers for Helmholtz
    return kx, jz, mh


def run_oracle_sample(cfg, repeats=1, shrink=1):
    """Times the oracle as it stands (Thomas / cyclic Thomas per line, OpenMP over lines). Returns (Gpts/s, info)."""
    sys.path.insert(0, os.path.join(ROOT, "oracle"))
    import oracle as orc
    from paper_1812_01178_b200 import inputs
    xf, yf, zf = cfg.faces()
    bcs = (orc.BC_DIRICHLET, orc.BC_DIRICHLET, orc.BC_PERIODIC)
    kx, jz, mh = (max(1, v // shrink) for v in sample_shapes(cfg))
    fxy = inputs.rhs_uniform((kx, cfg.ny, cfg.nx), cfg.seed)
    fz = inputs.rhs_uniform((cfg.nz, jz, cfg.nx), cfg.seed + 100)
    fh = inputs.rhs_complex_uniform((mh, cfg.ny, cfg.nx), cfg.seed)
    kz2 = cfg.kz2()[:mh]
    zf_k = np.linspace(0.0, 1.0, kx + 1) if kx >= 2 else np.array([0.0, 0.5, 1.0])
    yf_j = np.linspace(0.0, 1.0, jz + 1) if jz >= 2 else np.array([0.0, 0.5, 1.0])
    pts = 2 * fxy.size + fz.size + 2 * fh.size
    best = None
    for _ in range(repeats):
        t0 = time.perf_counter()
        orc.adi_sweep(fxy, xf, yf, zf_k, bcs, 0, orc.MODE_THOMAS, 1, cfg.alpha)
        orc.adi_sweep(fxy, xf, yf, zf_k, bcs, 1, orc.MODE_THOMAS, 1, cfg.alpha)
        orc.adi_sweep(fz, xf, yf_j, zf, bcs, 2, orc.MODE_THOMAS, 1, cfg.alpha)
        orc.helmholtz_solve(fh, yf, None, kz2, orc.MODE_THOMAS, 1)
        dt = time.perf_counter() - t0
        best = dt if best is None else min(best, dt)
    info = {"kind": "oracle", "cores": orc.num_threads(),
            "sample": "%s: x,y sweeps on %d z-planes, z sweep on %d y-rows, Helmholtz on %d wavenumbers (%.1f M real values, %.2f s)"
                      % (cfg.name, kx, jz, mh, pts / 1e6, best)}
    return pts / best / 1e9, best, info


def run_reference(args, rank, world):
    """--impl reference: the oracle on the host cores, each step a bounded sample of the workload (rank 0 only)."""
    if rank != 0:
        return
    cfg = configs.get(args.config)
    for _ in range(min(args.warmup, 1)):
        run_oracle_sample(cfg)
    times, val = [], None
    for _ in range(max(1, min(args.steps, 3))):
        val, dt, info = run_oracle_sample(cfg)
        times.append(dt)
    kx, jz, mh = sample_shapes(cfg)
    pts = 2 * kx * cfg.ny * cfg.nx + cfg.nz * jz * cfg.nx + 2 * mh * cfg.ny * cfg.nx
    t = float(np.mean(times))
    value = pts / t / 1e9
    info["value"] = value
    info["unit"] = UNIT
    print(json.dumps({"impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus,
                      "steps": len(times), "warmup": min(args.warmup, 1), "ms_per_step": t * 1e3, "higher_is_better": True,
                      "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
                      "config": {"workload": cfg.name + " (bounded sample per step)", "mode": "thomas (cpu oracle)"},
                      "cpu_baseline": info,
                      "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0}}))


def grid_table(tdx, torch, cfg_no, local_rank, steps, peak):
    """north_star: throughput on every BASELINE.json grid, per sweep direction, PPT and PDD, tuned P.  Fields that fit in
    L2 (cfg1, cfg2) are rotated through enough distinct copies to exceed 2 x L2, and still flagged informational (the
    launches are latency-bound there).  One event pair around each round of launches; Helmholtz right-hand sides are
    restored between rounds (that solve is not a contraction)."""
    cfg = configs.get(cfg_no)
    Ps = TUNED_P[cfg_no]
    bcs = (tdx.BC_DIRICHLET, tdx.BC_DIRICHLET, tdx.BC_PERIODIC)
    grid = tdx.Grid(cfg.nx, cfg.ny, cfg.nz, *cfg.faces(), bcs=bcs, device=local_rank)
    kz2 = cfg.kz2()
    stream = torch.cuda.current_stream().cuda_stream
    fbytes = cfg.npts * 8
    K = 1 if fbytes > 2 * 126e6 else int(min(16, -(-2 * 126e6 // fbytes)))   # cfg2: 8 copies = 2 x L2; cfg1 stays L2-resident (launch-bound anyway)
    f0 = torch.from_numpy(cfg.rhs_field()).cuda()
    h0 = torch.from_numpy(cfg.rhs_helmholtz()).cuda()
    fields = f0.unsqueeze(0).repeat(K, 1, 1, 1).contiguous()
    helms = h0.unsqueeze(0).repeat(K, 1, 1, 1).contiguous()
    names = ["adi_x", "adi_y", "adi_z_cyclic", "helmholtz_y"]
    pts = [cfg.npts, cfg.npts, cfg.npts, 2 * cfg.nx * cfg.ny * cfg.nm]
    out = {"grid": [cfg.nx, cfg.ny, cfg.nz], "points": cfg.npts, "copies_rotated": K,
           "l2": "larger than L2" if K == 1 else "field fits in L2, %d copies rotated (%.0f MB): GB/s informational" % (K, K * fbytes / 1e6)}
    rounds = max(3, steps // 2)
    for mname, mode in (("ppt", tdx.MODE_PPT), ("pdd", tdx.MODE_PDD)):
        res = {}
        for k, name in enumerate(names):
            if mname == "pdd" and k == 3:
                # PDD is not a valid solve for the Poisson y-systems (tests assert its error > 1e-3 on the
                # low modes): no throughput is quoted for it.  PPT is the production mode there, as in the paper.
                res[name] = {"skipped": "PDD is inaccurate on the weakly dominant Helmholtz systems (PAPER.md:L172): PPT only"}
                continue
            Pk, bound = Ps[k], None
            if mname == "pdd":
                Pk, bound = pdd_partitions(grid, cfg, k, Ps[k])
            def launch(c):
                if k < 3:
                    grid.adi_sweep(k, mode, Pk, cfg.alpha, fields[c], stream)
                else:
                    grid.helmholtz_wavenumber_solve(mode, Pk, None, kz2, helms[c], stream)
            for _ in range(3):
                for c in range(K):
                    launch(c)
            # Same protocol as the headline step: launches back to back on the stream between two events (REPS passes
            # over the K copies per event pair), so a figure is steady-state throughput and not one launch on an idle GPU
            # with its ramp-up and tail.  Sweeps run in place on their own output (same bytes; the Helmholtz right-hand
            # sides are restored before every round: that solve is not a contraction).
            REPS = 4
            tot = 0.0
            for _ in range(rounds):
                if k == 3:
                    helms.copy_(h0.unsqueeze(0).expand_as(helms))
                e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
                torch.cuda.synchronize()
                e0.record()
                for _rep in range(REPS):
                    for c in range(K):
                        launch(c)
                e1.record()
                torch.cuda.synchronize()
                tot += e0.elapsed_time(e1)
            ms = tot / (rounds * K * REPS)
            gbs = BYTES_PER_POINT * pts[k] / (ms * 1e-3) / 1e9
            res[name] = {"ms": ms, "gpts_per_s": pts[k] / (ms * 1e-3) / 1e9, "gb_per_s": gbs, "frac_of_measured_peak": gbs / peak,
                         "frac_of_nominal_8TBs": gbs / 8000.0, "P": Pk, "launch": tdx.last_launch()}
            if mname == "pdd":
                res[name]["dropped_bound"] = bound
                res[name]["pdd_gate_ok"] = bool(bound <= PDD_GATE)
        out[mname] = res
    if K > 1 or fbytes < 126e6:
        # Launch-bound grids: the whole step (x, y, cyclic z, Helmholtz; PPT) of all K copies captured ONCE in a CUDA graph
        # (the sweeps are plain stream work once their plans exist: no allocation, no synchronisation) and replayed.
        try:
            def step(c, st):
                for d in range(3):
                    grid.adi_sweep(d, tdx.MODE_PPT, Ps[d], cfg.alpha, fields[c], st)
                grid.helmholtz_wavenumber_solve(tdx.MODE_PPT, Ps[3], None, kz2, helms[c], st)
            side = torch.cuda.Stream()
            side.wait_stream(torch.cuda.current_stream())
            with torch.cuda.stream(side):
                for c in range(K):
                    step(c, side.cuda_stream)
                side.synchronize()
                n0 = tdx.kernel_launch_count()
                cg = torch.cuda.CUDAGraph()
                with torch.cuda.graph(cg, stream=side):
                    for c in range(K):
                        step(c, side.cuda_stream)
                captured = tdx.kernel_launch_count() - n0
            torch.cuda.synchronize()
            for _ in range(3):
                cg.replay()
            R = 50
            helms.copy_(h0.unsqueeze(0).expand_as(helms))
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            torch.cuda.synchronize()
            e0.record()
            for _ in range(R):
                cg.replay()
            e1.record()
            torch.cuda.synchronize()
            eager = sum(out["ppt"][n]["ms"] for n in names)
            out["step_cuda_graph"] = {"ms_per_step": e0.elapsed_time(e1) / (R * K), "eager_ms_per_step": eager, "kernels_in_graph": int(captured),
                                      "what": "x + y + cyclic z + Helmholtz (PPT) of the %d rotated copies captured in one CUDA graph, %d replays" % (K, R)}
            del cg
        except Exception as exc:                                 # an extra figure must never take the table down
            out["step_cuda_graph"] = {"error": repr(exc)[:300]}
    grid.close()
    del fields, helms, f0, h0
    return out


def run_tdx(args, rank, world, local_rank):
    import torch
    from paper_1812_01178_b200 import binding as tdx

    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device; the tdx path has no CPU fallback")
    torch.cuda.set_device(local_rank)
    dist = init_dist(world, "nccl", local_rank)
    cfg = configs.get(args.config)
    mode = {"ppt": tdx.MODE_PPT, "pdd": tdx.MODE_PDD, "thomas": tdx.MODE_THOMAS}[args.mode]
    Ps = tuple(int(v) for v in args.P.split(",")) if args.P else TUNED_P[args.config]
    bcs = (tdx.BC_DIRICHLET, tdx.BC_DIRICHLET, tdx.BC_PERIODIC)
    grid = tdx.Grid(cfg.nx, cfg.ny, cfg.nz, *cfg.faces(), bcs=bcs, device=local_rank)
    kz2 = cfg.kz2()
    # --mode pdd: the ADI sweeps run PDD with P chosen by rule (pdd_partitions: a-priori bound <= 1e-11, so north_star's
    # 1e-10 bar holds); the Poisson y-solves stay PPT -- PDD is not a valid solve there
    hmode, pdd_bounds = mode, [None, None, None]
    if args.mode == "pdd":
        hmode = tdx.MODE_PPT
        if not args.P:
            picked = [pdd_partitions(grid, cfg, d, Ps[d]) for d in range(3)]
            Ps = tuple(p for p, _ in picked) + (Ps[3],)
            pdd_bounds = [b for _, b in picked]
        else:
            pdd_bounds = [grid.pdd_dropped_bound(d, Ps[d], cfg.alpha) for d in range(3)]

    # inputs: seeded synthetic, generated once on the host, resident in HBM before the timed region
    host_field = cfg.rhs_field() if rank == 0 else None         # every rank solves its own field (weak scaling)
    if rank != 0:
        from paper_1812_01178_b200 import inputs
        host_field = inputs.rhs_uniform((cfg.nz, cfg.ny, cfg.nx), rank_seed(cfg, rank))
    host_helm = cfg.rhs_helmholtz()
    field0 = torch.from_numpy(host_field).cuda()
    helm0 = torch.from_numpy(host_helm).cuda()
    field = field0.clone()
    helm = helm0.clone()
    stream = torch.cuda.current_stream().cuda_stream

    launches_seen = []                                          # kernel instantiation + launch shape of the four sweeps

    def step(ev=None):
        # in place: re-running on its own output is the same work (same bytes); contraction keeps values bounded
        for k, d in enumerate((0, 1, 2)):
            if ev: ev[k].record()
            grid.adi_sweep(d, mode, Ps[d], cfg.alpha, field, stream)
            if launches_seen is not None and len(launches_seen) < 3: launches_seen.append(tdx.last_launch())
        if ev: ev[3].record()
        grid.helmholtz_wavenumber_solve(hmode, Ps[3], None, kz2, helm, stream)
        if launches_seen is not None and len(launches_seen) < 4: launches_seen.append(tdx.last_launch())
        if ev: ev[4].record()

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    for _ in range(max(args.warmup, 3)):
        step()
        helm.copy_(helm0)                                       # Helmholtz is not a contraction: restore its rhs
    barrier()
    evs = [[torch.cuda.Event(enable_timing=True) for _ in range(5)] for _ in range(args.steps)]
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    sampler = ClockSampler(local_rank)
    sampler.start()
    time.sleep(0.25)
    n0 = tdx.kernel_launch_count()
    barrier()
    e0.record()
    for s in range(args.steps):
        step(evs[s])
    e1.record()
    barrier()
    launches = tdx.kernel_launch_count() - n0
    sampler.stop_flag.set()
    total_ms = max_over_ranks(e0.elapsed_time(e1), dist, "cuda")
    ms_per_step = total_ms / args.steps
    value = whole_job_value(cfg, world, args.steps, total_ms)

    # per-kernel durations (CUDA events on the launching stream, inside the timed region)
    names = ["adi_x", "adi_y", "adi_z_cyclic", "helmholtz_y"]
    pts = [cfg.npts, cfg.npts, cfg.npts, 2 * cfg.nx * cfg.ny * cfg.nm]
    kms = [float(np.mean([evs[s][k].elapsed_time(evs[s][k + 1]) for s in range(args.steps)])) for k in range(4)]
    peak, peak_src = measured_peak()
    per_kernel = {n: {"ms": kms[k], "gpts_per_s": pts[k] / (kms[k] * 1e-3) / 1e9, "gb_per_s": BYTES_PER_POINT * pts[k] / (kms[k] * 1e-3) / 1e9,
                      "frac_of_measured_peak": BYTES_PER_POINT * pts[k] / (kms[k] * 1e-3) / 1e9 / peak,
                      "frac_of_nominal_8TBs": BYTES_PER_POINT * pts[k] / (kms[k] * 1e-3) / 1e9 / 8000.0, "P": Ps[k],
                      "launch": launches_seen[k] if k < len(launches_seen) else None} for k, n in enumerate(names)}
    for k in range(3):
        if pdd_bounds[k] is not None:
            per_kernel[names[k]]["dropped_bound"] = pdd_bounds[k]
            per_kernel[names[k]]["pdd_gate_ok"] = bool(pdd_bounds[k] <= PDD_GATE)
    if args.mode == "pdd":
        per_kernel[names[3]]["mode"] = "ppt (PDD is not a valid solve for the Poisson y-systems, PAPER.md:L172)"
    dom = int(np.argmax(kms))
    achieved = BYTES_PER_POINT * pts[dom] / (kms[dom] * 1e-3) / 1e9
    traffic, traffic_src = ncu_traffic(cfg.name, per_kernel[names[dom]]["launch"])
    roofline = {"bound": "hbm", "kernel": names[dom], "launch": per_kernel[names[dom]]["launch"], "achieved": achieved, "peak": peak,
                "unit": "GB/s", "frac": achieved / peak, "traffic": traffic, "traffic_source": traffic_src,
                "peak_source": peak_src, "algorithmic_bytes_per_launch": BYTES_PER_POINT * pts[dom],
                "share_of_step": kms[dom] / sum(kms)}

    out = {"metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": max(args.warmup, 3),
           "ms_per_step": ms_per_step, "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64",
           "data": "synthetic",
           "config": {"workload": cfg.name, "grid": [cfg.nx, cfg.ny, cfg.nz], "mode": args.mode,
                      "P": {"x": Ps[0], "y": Ps[1], "z": Ps[2], "helmholtz": Ps[3]}, "alpha": cfg.alpha, "nm": cfg.nm,
                      "step": "adi x + adi y + adi z (cyclic) + helmholtz y-solves, in place",
                      "l2": "inputs larger than L2 (%.2f GB field, %.2f GB complex)" % (cfg.npts * 8 / 1e9, cfg.nx * cfg.ny * cfg.nm * 16 / 1e9)
                      if cfg.npts * 8 > 2 * 126e6 else "L2-resident field: GB/s informational only",
                      "parallelism": "independent field per GPU, no collective"},
           "kernels": per_kernel, "roofline": roofline, "gpu_launches": int(launches), "clocks": sampler.summary()}

    # one tdx_adi_step over three staggered velocity components stored back to back (u: face in x,
    # v: face in y, w: face in z), x -> y -> z, 3 launches.  Reported beside the headline, not part of `value`.
    if not args.no_step3 and torch.cuda.mem_get_info()[0] > 3.3 * cfg.npts * 8:
        comps = field0.unsqueeze(0).repeat(3, 1, 1, 1).contiguous()
        locs = [[1, 0, 0], [0, 1, 0], [0, 0, 1]]
        for _ in range(3):
            grid.adi_step(mode, Ps[0], Ps[1], Ps[2], cfg.alpha, 3, locs, comps, stream)
        barrier()
        s0, s1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        s0.record()
        for _ in range(args.steps):
            grid.adi_step(mode, Ps[0], Ps[1], Ps[2], cfg.alpha, 3, locs, comps, stream)
        s1.record()
        barrier()
        ms3 = max_over_ranks(s0.elapsed_time(s1) / args.steps, dist, "cuda")
        out["adi_step_3comp"] = {"ms": ms3, "gpts_per_s": 9 * cfg.npts / (ms3 * 1e-3) / 1e9,
                                 "gb_per_s": BYTES_PER_POINT * 9 * cfg.npts / (ms3 * 1e-3) / 1e9,
                                 "frac_of_measured_peak": BYTES_PER_POINT * 9 * cfg.npts / (ms3 * 1e-3) / 1e9 / peak,
                                 "what": "tdx_adi_step: 3 staggered components x (x, y, z) sweeps, 9 field sweeps in 3+ launches"}
        del comps

    # Helmholtz y-solves with a different shift per line (lambda = kx'^2(i) + kz'^2(m), the paper's
    # cosine-x / Fourier-z Poisson solve): factorisation, spikes and reduced system on the fly.  The call synchronises
    # (kx2/kz2 are host arrays), so these times include one host round trip.  Reported beside the headline.
    if not args.no_step3:
        from paper_1812_01178_b200 import inputs as _inp
        kx2 = _inp.modified_wavenumbers_x(cfg.nx, cfg.lx)
        Pl = TUNED_P_LINE[args.config]
        per_line = {}
        for mname, mval in (("ppt", tdx.MODE_PPT), ("pdd", tdx.MODE_PDD)):
            helm.copy_(helm0)
            for _ in range(2):
                grid.helmholtz_wavenumber_solve(mval, Pl, kx2, kz2, helm, stream)
            barrier()
            s0, s1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            s0.record()
            for _ in range(args.steps):
                grid.helmholtz_wavenumber_solve(mval, Pl, kx2, kz2, helm, stream)
            s1.record()
            barrier()
            msl = max_over_ranks(s0.elapsed_time(s1) / args.steps, dist, "cuda")
            per_line[mname] = {"ms": msl, "gb_per_s": BYTES_PER_POINT * pts[3] / (msl * 1e-3) / 1e9, "P": Pl}
        out["helmholtz_per_line_shift"] = per_line

        # the whole direct Poisson solve: cosine-x, Fourier-z, per-line y-solves, inverse
        # transforms -- five passes over the field; per-pass times from events around the single-stage entry points.
        del helm
        work = helm0                                             # spectrum scratch (its right-hand side is no longer needed)
        pfield = field0.clone()
        stages = [("dct_x", lambda: grid.dct_x(False, pfield, stream), BYTES_PER_POINT * cfg.npts),
                  ("rfft_z", lambda: grid.rfft_z(pfield, work, stream), 8 * cfg.npts + 16 * cfg.nx * cfg.ny * cfg.nm),
                  ("irfft_z", lambda: grid.irfft_z(work, pfield, stream), 8 * cfg.npts + 16 * cfg.nx * cfg.ny * cfg.nm),
                  ("idct_x", lambda: grid.dct_x(True, pfield, stream), BYTES_PER_POINT * cfg.npts)]
        pstage = {}
        for sname, fn, nbytes in stages:
            for _ in range(3):
                fn()
            barrier()
            s0, s1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            s0.record()
            for _ in range(args.steps):
                fn()
            s1.record()
            barrier()
            mst = max_over_ranks(s0.elapsed_time(s1) / args.steps, dist, "cuda")
            pstage[sname] = {"ms": mst, "gb_per_s": nbytes / (mst * 1e-3) / 1e9, "frac_of_measured_peak": nbytes / (mst * 1e-3) / 1e9 / peak}
        pfield.copy_(field0)
        for _ in range(2):
            grid.poisson_solve(tdx.MODE_PPT, Pl, None, None, pfield, work, stream)
        barrier()
        s0, s1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        s0.record()
        for _ in range(args.steps):
            grid.poisson_solve(tdx.MODE_PPT, Pl, None, None, pfield, work, stream)
        s1.record()
        barrier()
        msp = max_over_ranks(s0.elapsed_time(s1) / args.steps, dist, "cuda")
        out["poisson_solve"] = {"ms": msp, "gpts_per_s": cfg.npts / (msp * 1e-3) / 1e9, "mode": "ppt", "P": Pl,
                                "algorithmic_bytes": 5 * BYTES_PER_POINT * cfg.npts,
                                "gb_per_s": 5 * BYTES_PER_POINT * cfg.npts / (msp * 1e-3) / 1e9,
                                "frac_of_measured_peak": 5 * BYTES_PER_POINT * cfg.npts / (msp * 1e-3) / 1e9 / peak,
                                "stages": pstage,
                                "what": "tdx_poisson_solve: dct_x, rfft_z, per-line y-solves (PPT), irfft_z, idct_x; 80 B per grid value"}
        del pfield, work

        # per-line coefficients with diagonal pivoting along y -- the partition method with pivoted local
        # solves, one pass: a, b, c, d in, x out = 40 algorithmic bytes per value.  Two workloads: the paper's own case
        # (L172-174: weakly dominant Poisson-like rows |b| = |a| + |c| + eps, eps differing from line to line, handed over
        # as explicit coefficients), where no line leaves the partition kernel, and random NON-dominant systems
        # (|b| <= 0.3, |a|, |c| <= 1), where every line with a numerically singular 8-row block is re-solved by the
        # per-line path (their share is reported).
        try:
            if torch.cuda.mem_get_info()[0] > 6.5 * cfg.npts * 8:
                gen = torch.Generator(device=field0.device); gen.manual_seed(1234)
                ga, gc = (torch.rand(field0.shape, dtype=torch.float64, device=field0.device, generator=gen) * 2 - 1 for _ in range(2))
                gb = (torch.rand(field0.shape, dtype=torch.float64, device=field0.device, generator=gen) * 2 - 1) * 0.3
                gd = field0.clone()
                gwork = torch.empty(9 * cfg.npts + 64, dtype=torch.uint8, device=field0.device)
                gout = {}
                for wname in ("poisson_like_weakly_dominant", "random_non_dominant"):
                    if wname == "poisson_like_weakly_dominant":
                        ga.abs_().add_(0.2).neg_(); gc.abs_().add_(0.2).neg_()
                        ga[:, 0, :] = 0.0; gc[:, -1, :] = 0.0
                        eps = torch.pow(10.0, -6.0 * gb[:, :1, :].abs() / 0.3)          # one shift per line, 1e-6 ... 1
                        gb = -(ga + gc) + eps
                        del eps
                    else:
                        ga, gc = (torch.rand(field0.shape, dtype=torch.float64, device=field0.device, generator=gen) * 2 - 1 for _ in range(2))
                        gb = (torch.rand(field0.shape, dtype=torch.float64, device=field0.device, generator=gen) * 2 - 1) * 0.3
                    res = {}
                    # both methods (include/tdx.h): "partition" = the one-pass partition kernel (the default: optimistic plain
                    # elimination inside the partitions, checked, unsafe lines re-solved with pivots); "lines" = one thread
                    # per line with diagonal pivoting, two passes
                    # "default" = no method forced: a sample of the rows decides on the device (mostly non-dominant rows: the
                    # per-line kernel on every line; else the partition kernel)
                    for meth, flag, nbytes in (("lines", tdx.GENERAL_FORCE_LINES, 82), ("partition", tdx.GENERAL_FORCE_PARTITION, 40), ("default", 0, 40)):
                        for _ in range(2):
                            gd.copy_(field0); grid.general_solve(1, 1 | flag, ga, gb, gc, gd, gwork, stream)
                        barrier()
                        tot = 0.0
                        for _ in range(args.steps):
                            gd.copy_(field0)
                            s0, s1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
                            s0.record(); grid.general_solve(1, 1 | flag, ga, gb, gc, gd, gwork, stream); s1.record()
                            torch.cuda.synchronize()
                            tot += s0.elapsed_time(s1)
                        msg = max_over_ranks(tot / args.steps, dist, "cuda")
                        nfb = grid.general_fallback_count()
                        launch = tdx.last_launch()
                        if meth == "default" and nfb == cfg.nx * cfg.nz:
                            nbytes = 82                                    # the device chose the per-line kernel for every line
                            launch = "k_general_lines<1,0,0> on every line (chosen on the device; the partition kernel returned at once)"
                        res[meth] = {"ms": msg, "gpts_per_s": cfg.npts / (msg * 1e-3) / 1e9, "algorithmic_bytes_per_value": nbytes,
                                     "gb_per_s": nbytes * cfg.npts / (msg * 1e-3) / 1e9,
                                     "frac_of_measured_peak": nbytes * cfg.npts / (msg * 1e-3) / 1e9 / peak, "finite": bool(torch.isfinite(gd).all()),
                                     "lines_re_solved_by_the_per_line_kernel": nfb, "share_of_lines": nfb / (cfg.nx * cfg.nz), "launch": launch}
                    gout[wname] = res
                gout["what"] = ("tdx_general_solve along y, per-line a, b, c, diagonal pivoting: partition kernel (8-row partitions, one pass, 40 B per value), "
                                "per-line kernel (two passes, 82 B per value), and the default (the device picks one of the two from a sample of the rows)")
                out["general_solve_pivoting"] = gout
                del ga, gb, gc, gd, gwork
        except Exception as exc:
            out["general_solve_pivoting"] = {"error": repr(exc)[:300]}

        # the y sweep with the field cut into y-slabs, one per rank (the paper's decomposition, L74): local
        # elimination (the slab's own sweep kernel) + interface exchange + one correction pass = 32 B per grid value.
        # world == 1: the compute part of an interior rank of a 4-rank job (a quarter slab; the exchange is a device copy);
        # world > 1: the real thing over NCCL (strong scaling of ONE field), max over ranks.
        try:
            if args.no_slab:
                raise RuntimeError("skipped (--no-slab)")
            from paper_1812_01178_b200 import parallel
            Rk = world if world > 1 else 4
            rk = rank if world > 1 else 1
            y0, y1 = parallel.slab_bounds(cfg.ny, Rk)[rk]
            fs = cfg.faces()
            sg = tdx.Grid(cfg.nx, y1 - y0, cfg.nz, fs[0], fs[1][y0:y1 + 1], fs[2], bcs=bcs, device=local_rank)
            Ploc = max(p for p in range(1, (y1 - y0) // 2 + 1) if (y1 - y0) % p == 0 and (y1 - y0) // p >= 8) if (y1 - y0) >= 16 else 1
            slab_out = {"ranks": Rk, "rows_per_rank": y1 - y0, "P_local": Ploc}
            sfield = field0[:, y0:y1, :].contiguous()
            for aname, across in (("ppt", tdx.MODE_PPT), ("pdd", tdx.MODE_PDD)):
                sw = parallel.SlabSweep(sg, 1, rk, Rk, fs[1], bcs[1], cfg.alpha, across, tdx.MODE_PPT if Ploc > 1 else tdx.MODE_THOMAS, Ploc)
                if world > 1:
                    run = lambda: sw.sweep(sfield)
                else:
                    iface = torch.zeros((2, cfg.nx * cfg.nz), dtype=torch.float64, device=sfield.device)
                    gathered = torch.zeros((Rk, 2, cfg.nx * cfg.nz), dtype=torch.float64, device=sfield.device)
                    def run():
                        sw.slab.eliminate(sfield, iface, stream)
                        gathered[rk].copy_(iface)                # stands in for the exchange
                        sw.slab.correct(sfield, iface, gathered if across == tdx.MODE_PPT else gathered[rk], stream)
                for _ in range(3):
                    run()
                barrier()
                s0, s1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
                s0.record()
                for _ in range(args.steps):
                    run()
                s1.record()
                barrier()
                mss = max_over_ranks(s0.elapsed_time(s1) / args.steps, dist, "cuda")
                npt = cfg.npts if world > 1 else sfield.numel()
                slab_out[aname] = {"ms": mss, "gpts_per_s": npt / (mss * 1e-3) / 1e9, "gb_per_s": 2 * BYTES_PER_POINT * npt / (mss * 1e-3) / 1e9 / (world if world > 1 else 1),
                                   "dropped_bound": sw.slab.dropped_bound()}
                sw.close()
            slab_out["what"] = ("y sweep of the whole field over %d ranks (NCCL exchange), whole-job Gpts/s, per-GPU GB/s at 32 B/value" % world) if world > 1 else \
                               "compute part of one interior rank of a 4-rank y-slab sweep (eliminate + correct, exchange replaced by a device copy)"
            out["slab_y_sweep"] = slab_out
            sg.close()
            del sfield
        except Exception as exc:                                 # an extra figure must never take the headline down
            out["slab_y_sweep"] = {"error": repr(exc)[:300]}

    # north_star: "throughput on the five synthetic grids ... per sweep direction and as a fraction of the HBM roofline":
    # the other BASELINE.json grids beside the headline one (same kernels, their own tuned P), rank 0 at N = 1 only.
    if not args.no_step3 and world == 1:
        try:
            torch.cuda.empty_cache()
            out["grids"] = {configs.get(c).name: grid_table(tdx, torch, c, local_rank, args.steps, peak)
                            for c in (1, 2, 3, 4, 5) if c != args.config}
        except Exception as exc:                                 # an extra figure must never take the headline down
            out["grids"] = {"error": repr(exc)[:300]}

    # end to end through the host-buffer C-ABI calls: pinned host buffers, H2D + solve + D2H inside the timed region
    if not args.no_e2e and hmode != mode:
        out["e2e"] = {"skipped": "tdx_step_host runs one mode for the whole step; the end-to-end figure is quoted for --mode ppt"}
    elif not args.no_e2e:
        # two independent pinned buffer pairs: consecutive steps go through tdx_step_host_async in alternating slots, so one
        # step's download runs beside the next step's upload (one call alone is bound to three transfer times)
        pairs, two = [], 1.0
        try:
            for _ in range(2):
                pairs.append((torch.from_numpy(host_field).pin_memory().numpy(), torch.from_numpy(host_helm).pin_memory().numpy()))
        except RuntimeError:                                                       # no room to page-lock a second pair on this host
            two = 0.0
        two = -max_over_ranks(-two, dist, "cuda") > 0.5                            # every rank or none
        nslots = 2 if two else 1
        hf, hh = pairs[0]
        grid.step_host(mode, Ps[0], Ps[1], Ps[2], cfg.alpha, hf, Ps[3], kz2, hh)   # warm-up (staging allocation, streams)
        np.copyto(hh, host_helm)
        barrier()
        t0 = time.perf_counter()                                                   # one synchronous call on its own
        grid.step_host(mode, Ps[0], Ps[1], Ps[2], cfg.alpha, hf, Ps[3], kz2, hh)
        torch.cuda.synchronize()
        t_single = time.perf_counter() - t0
        for slot in range(nslots):                                                 # warm-up of the second slot's staging
            grid.step_host_async(slot, mode, Ps[0], Ps[1], Ps[2], cfg.alpha, pairs[slot][0], Ps[3], kz2, pairs[slot][1])
        for slot in range(nslots):
            grid.step_host_wait(slot)
        for slot in range(nslots):
            np.copyto(pairs[slot][1], host_helm)
        nsteps = max(8, 2 * args.e2e_steps)                                        # fill and drain cost one transfer time in all
        barrier()
        t0 = time.perf_counter()
        for k in range(nsteps):
            slot = k % nslots
            if k >= nslots:
                grid.step_host_wait(slot)                                          # the step that used this slot's buffers is home
            grid.step_host_async(slot, mode, Ps[0], Ps[1], Ps[2], cfg.alpha, pairs[slot][0], Ps[3], kz2, pairs[slot][1])
        for slot in range(nslots):
            grid.step_host_wait(slot)
        torch.cuda.synchronize()
        te = max_over_ranks((time.perf_counter() - t0) / nsteps, dist, "cuda")
        t_single = max_over_ranks(t_single, dist, "cuda")
        out["e2e"] = {"value": world * step_points(cfg) / te / 1e9, "unit": UNIT, "h2d_bytes_per_step": int(hf.nbytes + hh.nbytes),
                      "d2h_bytes_per_step": int(hf.nbytes + hh.nbytes), "ms_per_step": te * 1e3, "steps": nsteps,
                      "single_call_ms": t_single * 1e3, "single_call_value": world * step_points(cfg) / t_single / 1e9,
                      "steps_in_flight": nslots,
                      "api": "tdx_step_host_async / tdx_step_host_wait, two steps in flight on two pinned buffer pairs (every step's "
                             "inputs go up and its results come down inside the timed region); single_call = one synchronous "
                             "tdx_step_host"}
    if rank == 0 and world == 1 and not args.no_cpu:
        v, _, info = run_oracle_sample(cfg)
        info["value"] = v
        info["unit"] = UNIT
        try:                                                       # a 1-thread figure beside it (an eighth of the sample)
            sys.path.insert(0, os.path.join(ROOT, "oracle"))
            import oracle as orc
            ncores = orc.num_threads()
            orc.set_num_threads(1)
            v1, _, info1 = run_oracle_sample(cfg, shrink=8)
            orc.set_num_threads(ncores)
            info["value_1_thread"] = v1
            info["sample_1_thread"] = info1["sample"]
        except Exception as exc:
            info["value_1_thread"] = None
            info["sample_1_thread"] = repr(exc)[:200]
        out["cpu_baseline"] = info
    grid.close()
    if world > 1:
        out["nccl"] = nccl_log_summary()
        out["nccl_comm_nranks_ok"] = bool(out["nccl"] and world in out["nccl"].get("nranks_seen", []))
    if rank == 0:
        print(json.dumps(out))
    if world > 1:
        dist.destroy_process_group()


def run_psweep(args):
    """BASELINE.json config 3's purpose: PDD vs PPT over P -- throughput and accuracy per sweep direction."""
    import torch
    sys.path.insert(0, os.path.join(ROOT, "oracle"))
    import oracle as orc
    from paper_1812_01178_b200 import binding as tdx
    cfg = configs.get(args.config)
    bcs = (tdx.BC_DIRICHLET, tdx.BC_DIRICHLET, tdx.BC_PERIODIC)
    faces = cfg.faces()
    grid = tdx.Grid(cfg.nx, cfg.ny, cfg.nz, *faces, bcs=bcs)
    field0 = torch.from_numpy(cfg.rhs_field()).cuda()
    rng = np.random.default_rng(7)
    ns = 48
    print("| dir | mode | P | rows/partition | ms | GB/s | PDD dropped bound | rel. error of %d sampled lines vs oracle | launch |" % ns)
    print("|---|---|---|---|---|---|---|---|---|")
    for d, name in enumerate("xyz"):
        n = (cfg.nx, cfg.ny, cfg.nz)[d]
        dims = {0: (cfg.nz, cfg.ny), 1: (cfg.nz, cfg.nx), 2: (cfg.ny, cfg.nx)}[d]
        ia = torch.from_numpy(rng.integers(0, dims[0], ns)).cuda(); ib = torch.from_numpy(rng.integers(0, dims[1], ns)).cuda()
        take = {0: lambda t: t[ia, ib, :], 1: lambda t: t[ia, :, ib], 2: lambda t: t[:, ia, ib].t()}[d]
        a, b, c = orc.adi_coeffs(faces[d], bcs[d], cfg.alpha)
        solve = orc.cyclic_thomas if bcs[d] == orc.BC_PERIODIC else orc.thomas
        ref = np.stack([solve(a, b, c, row) for row in take(field0).cpu().numpy()])
        for mode_name, mode in (("pdd", tdx.MODE_PDD), ("ppt", tdx.MODE_PPT)):
            for P in [int(v) for v in args.psweep.split(",")]:
                if n // P < 2:
                    continue
                try:
                    t = field0.clone()
                    grid.adi_sweep(d, mode, P, cfg.alpha, t)
                    torch.cuda.synchronize()
                    err = float(np.max(np.abs(take(t).cpu().numpy() - ref)) / np.max(np.abs(ref)))
                    for _ in range(3):
                        grid.adi_sweep(d, mode, P, cfg.alpha, t)
                    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
                    torch.cuda.synchronize(); e0.record()
                    for _ in range(10):
                        grid.adi_sweep(d, mode, P, cfg.alpha, t)
                    e1.record(); torch.cuda.synchronize()
                    ms = e0.elapsed_time(e1) / 10
                    drop = grid.pdd_dropped_bound(d, P, cfg.alpha)
                    print("| %s | %s | %d | %d | %.3f | %.0f | %.1e | %.1e | `%s` |" % (name, mode_name, P, -(-n // P), ms, BYTES_PER_POINT * cfg.npts / ms / 1e6, drop, err, tdx.last_launch()))
                except tdx.TdxError as e:
                    print("| %s | %s | %d | %d | - | - | - | %s | - |" % (name, mode_name, P, -(-n // P), tdx.status_string(e.status)))
    grid.close()


def main():
    args = parse()
    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local_rank = int(os.environ.get("LOCAL_RANK", "0"))
    if args.psweep:
        if rank == 0:
            run_psweep(args)
    elif args.selftest_ranks:
        selftest_ranks(args, rank, world)
    elif args.impl == "reference":
        run_reference(args, rank, world)
    else:
        run_tdx(args, rank, world, local_rank)


if __name__ == "__main__":
    main()
