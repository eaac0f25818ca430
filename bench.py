"""bench.py — tendency+RK3 cell-updates/s of the hot path on the B200 (BASELINE.json metric).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--workload C2] [--impl ours|reference]

One *step* = one full RK3 time step of the workload = 3 substages, each {ocn_fill_halos, [C3: ocn_compute_w,
ocn_compute_phy], ocn_compute_tendencies, ocn_rk3_substage} through the C ABI of libocn.so, on seeded synthetic
fields resident in HBM.  value = Nx*Ny*Nz*3*K*N / elapsed (cell-updates/s, whole job).  The default workload is
C2 (512x512x256 fp64, the configuration the north_star's roofline target is quoted on; every field is 562 MB,
far larger than the 126 MB L2, so no flush is needed between iterations).

  * `e2e`      : the same metric through ocn_step_host (pinned HOST buffers in, HOST buffers out, copies timed).
  * `roofline` : the fused tendency kernel, compulsory bytes per launch / its CUDA-event duration measured inside
                 the timed region, against the measured HBM copy peak of MEASURED_PEAKS.json.
  * `cpu_baseline` : the CPU oracle (as it stands) on the box's host cores on a bounded sample (rank 0, N=1).
  * `--impl reference` times that oracle instead of the CUDA path (there is no reference implementation).
N > 1 (torchrun): independent replicas of the same workload, one per GPU ("replicas only": the north_star fixes
the path to one GPU), barrier + max over ranks.
"""
import argparse
import json
import os
import subprocess
import sys
import threading
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

METRIC = "tendency+RK3 cell-updates/sec"
UNIT = "cell-updates/s"
CPU_SAMPLE = {"C0": None, "C1": (128, 128, 32), "C2": (256, 256, 32), "C3": (360, 150, 50), "C4": (256, 256, 32)}


def _peaks():
    try:
        with open(os.path.join(ROOT, "MEASURED_PEAKS.json")) as f:
            p = json.load(f)
        return float(p["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs)"
    except Exception:
        return 6650.0, "fallback (B200_PROFILING.md 6.65 TB/s)"


class ClockSampler:
    """nvidia-smi clocks / throttle reasons DURING the timed region (B200_PROFILING.md 'clocks line')."""
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,"
         "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")

    def __init__(self, index):
        self.rows, self.p, self.index = [], None, index

    def start(self):
        try:
            self.p = subprocess.Popen(["nvidia-smi", "-i", str(self.index), "--query-gpu=" + self.Q,
                                       "--format=csv,noheader,nounits", "-lms", "100"],
                                      stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            self.t = threading.Thread(target=self._read, daemon=True)
            self.t.start()
        except Exception:
            self.p = None

    def _read(self):
        for line in self.p.stdout:
            self.rows.append([x.strip() for x in line.split(",")])

    def stop(self):
        if self.p is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        time.sleep(0.15)
        self.p.terminate()
        try:
            self.p.wait(timeout=5)
        except Exception:
            self.p.kill()
        sm, mx, reasons = [], None, set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for r in self.rows:
            try:
                sm.append(float(r[0])); mx = float(r[1])
                for n, v in zip(names, r[3:7]):
                    if v.lower().startswith("active"):
                        reasons.add(n)
            except Exception:
                pass
        sm.sort()
        return {"sm_mhz": sm[len(sm) // 2] if sm else None, "sm_max_mhz": mx, "reasons": sorted(reasons), "samples": len(sm)}


def compulsory_bytes(cfg, lay_elems_padded):
    """tendency kernel: every input field read once + every output field written once, halos included
    (north_star): inputs over the padded extents, outputs over the interior."""
    p, g = cfg["params"], cfg["grid"]
    esz = 8 if cfg["dtype"] == "f64" else 4
    interior = g["Nx"] * g["Ny"] * g["Nz"]
    n_in = p["n_tracers"] + (2 if g["topology"][2] == 2 else 3) + (1 if p["hydrostatic"] else 0)
    n_out = p["n_tracers"] + (0 if not p["momentum_prognostic"] else (2 if (p["hydrostatic"] or g["topology"][2] == 2) else 3))
    return esz * (n_in * lay_elems_padded + n_out * interior), n_in, n_out


def cpu_oracle_leg(name, steps=1, warmup=0):
    """the oracle (double / float instantiation, OpenMP over the host cores) on a bounded sample of the workload:
    the same recipe on a sub-grid, `steps` full RK3 steps.  Returns (cell-updates/s, cores, sample text, seconds)."""
    from oracle import ocnref as ref
    from paper_2502_14148_b200 import workloads as W
    size = CPU_SAMPLE[name]
    cfg = W.get_config(name, size=size)
    g = cfg["grid"]
    state = W.generate_state(cfg)
    rg = ref.RefGrid(g["Nx"], g["Ny"], g["Nz"], g["halo"], g["dx"], g["dy"], g["dz_c"], g["dz_uniform"], g["topology"])
    for _ in range(warmup):
        ref.step(rg, cfg["params"], 3, cfg["dt"], state, eval=1)
    t0 = time.perf_counter()
    for _ in range(steps):
        ref.step(rg, cfg["params"], 3, cfg["dt"], state, eval=1)
    dt = time.perf_counter() - t0
    cells = g["Nx"] * g["Ny"] * g["Nz"]
    sample = "%s recipe on a %dx%dx%d sub-grid, %d full RK3 step(s) (3 substages each), %s evaluation" % (
        name, g["Nx"], g["Ny"], g["Nz"], steps, "double" if cfg["dtype"] == "f64" else "float")
    return cells * 3 * steps / dt, ref.num_threads(), sample, dt, cfg


def reference_arm(args, rank, world):
    """--impl reference: there is no reference implementation (the paper ships no code); the arm is the CPU
    oracle, as it stands, timed on the host cores on a bounded sample of the same workload.  Rank 0 only."""
    if rank != 0:
        return
    steps = max(1, min(args.steps, 2))
    warm = 1 if args.warmup > 0 else 0
    v, cores, sample, dt, cfg = cpu_oracle_leg(args.workload, steps=steps, warmup=warm)
    g = cfg["grid"]
    line = {"impl": "reference", "metric": METRIC, "value": v, "unit": UNIT, "n_gpus": world, "steps": steps, "warmup": warm,
            "ms_per_step": 1e3 * dt / steps, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
            "dtype": cfg["dtype"], "data": "synthetic",
            "config": {"workload": "%s (%s)" % (args.workload, cfg["description"]), "sample_grid": [g["Nx"], g["Ny"], g["Nz"]],
                       "substages_per_step": 3},
            "cpu_baseline": {"value": v, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": sample},
            "e2e": {"value": v, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0}
    print(json.dumps(line), flush=True)


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=10)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--workload", default="C2", choices=["C0", "C1", "C2", "C3", "C4"])
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--kernel", type=int, default=0, help="0 auto (fused where it applies), 1 per-cell, 2 fused")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-e2e", action="store_true")
    args = ap.parse_args()
    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if args.impl == "reference":
        return reference_arm(args, rank, world)
    if args.warmup < 3:
        args.warmup = 3     # timing rule: W >= 3

    import torch
    import torch.distributed as dist
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device — the product path has no CPU fallback")
    torch.cuda.set_device(local)
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))
    from paper_2502_14148_b200 import binding as B, workloads as W
    B.lib()

    cfg = W.get_config(args.workload)
    p, g = cfg["params"], cfg["grid"]
    hydro = bool(p["hydrostatic"])
    dev = torch.device("cuda", local)
    grid = B.ocn_grid_create(g["Nx"], g["Ny"], g["Nz"], g["halo"], g["dx"], g["dy"], g["dz_c"], g["dz_uniform"],
                             g["topology"], cfg["dtype"], device=dev)
    grid.set_kernel(args.kernel)
    big = g["Nx"] * g["Ny"] * g["Nz"] > 4_000_000
    state0 = W.generate_state(cfg, device=dev if big else "cpu", as_numpy=False)
    st = grid.fields_from_state(state0)
    del state0
    torch.cuda.empty_cache()
    hasw = g["topology"][2] != 2 and not hydro
    mom = bool(p["momentum_prognostic"])
    mkG = lambda: grid.fields(n_tracers=p["n_tracers"], u=mom, v=mom, w=mom and hasw)
    G, Gp = mkG(), mkG()
    phy = grid.new_field() if hydro else None
    cp = B.make_params(p)
    dt = cfg["dt"]
    cells = g["Nx"] * g["Ny"] * g["Nz"]
    L = grid.layout
    padded = L.nx_pad * L.ny_pad * L.nz_pad
    tb, n_in, n_out = compulsory_bytes(cfg, padded)

    def substage(m, Gm, Gq, ev=None):
        B.ocn_fill_halos(grid, cp, st)
        if hydro:
            B.ocn_compute_w(grid, st)
            B.ocn_compute_phy(grid, cp, st, phy)
        if ev is not None:
            ev[0].record()
        B.ocn_compute_tendencies(grid, cp, st, phy, Gm)
        if ev is not None:
            ev[1].record()
        B.ocn_rk3_substage(grid, cp, m, dt, st, Gm, None if m == 1 else Gq)

    def step(evs=None):
        a, b = G, Gp
        for m in (1, 2, 3):
            substage(m, a, b, None if evs is None else evs[m - 1])
            a, b = b, a

    def sync():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    for _ in range(args.warmup):
        step()
    K = args.steps
    evs = [[(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(3)] for _ in range(K)]
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    sampler = ClockSampler(local)
    sampler.start()
    sync()
    n0 = B.ocn_launch_count()
    e0.record()
    for k in range(K):
        step(evs[k])
    e1.record()
    sync()
    launches = B.ocn_launch_count() - n0
    clocks = sampler.stop()
    ms = e0.elapsed_time(e1)
    tend_ms = [a.elapsed_time(b) for row in evs for (a, b) in row]
    if world > 1:
        t = torch.tensor([ms], device=dev, dtype=torch.float64)
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
        ms = float(t.item())
    value = cells * 3 * K * world / (ms * 1e-3)
    tend_avg = sum(tend_ms) / len(tend_ms)
    finite = all(bool(torch.isfinite(t).all()) for t in st.all())

    # ---- per-call breakdown (diagnostic pass after the timed region; not part of `value`)
    def timed(fn, n=3):
        a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        torch.cuda.synchronize(); a.record()
        for _ in range(n):
            fn()
        b.record(); torch.cuda.synchronize()
        return a.elapsed_time(b) / n
    breakdown = {"fill_halos": timed(lambda: B.ocn_fill_halos(grid, cp, st)),
                 "tendencies": tend_avg,
                 "rk3_substage_stage1": timed(lambda: B.ocn_substage(grid, cp, 0.0, 0.0, dt, st, G, None)),
                 "rk3_substage_stage23": timed(lambda: B.ocn_substage(grid, cp, 0.0, 1e-300, dt, st, G, Gp))}
    if hydro:
        breakdown["compute_w"] = timed(lambda: B.ocn_compute_w(grid, st))
        breakdown["compute_phy"] = timed(lambda: B.ocn_compute_phy(grid, cp, st, phy))

    # ---- end to end: HOST buffers in, HOST buffers out, through ocn_step_host
    e2e = None
    if not args.no_e2e:
        host = B.Fields(*[None if t is None else torch.empty_like(t, device="cpu").pin_memory() for t in (st.u, st.v, st.w)],
                        [torch.empty_like(t, device="cpu").pin_memory() for t in st.c])
        for h, d in zip(host.all(), st.all()):
            h.copy_(d)
        esz = 8 if cfg["dtype"] == "f64" else 4
        nf_in = len(host.all())
        nf_out = (p["n_tracers"] + ((3 if hasw else 2) if mom else 0))
        Ke = max(1, min(K, 3))
        B.ocn_step_host(grid, cp, 3, dt, host, st, G, Gp, phy)      # warm-up
        sync()
        a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        a.record()
        for _ in range(Ke):
            B.ocn_step_host(grid, cp, 3, dt, host, st, G, Gp, phy)
        b.record()
        sync()
        ems = a.elapsed_time(b)
        if world > 1:
            t = torch.tensor([ems], device=dev, dtype=torch.float64)
            dist.all_reduce(t, op=dist.ReduceOp.MAX)
            ems = float(t.item())
        e2e = {"value": cells * 3 * Ke * world / (ems * 1e-3), "unit": UNIT, "h2d_bytes_per_step": nf_in * L.n_alloc * esz,
               "d2h_bytes_per_step": nf_out * L.n_alloc * esz, "steps": Ke, "ms_per_step": ems / Ke,
               "api": "ocn_step_host (pinned host buffers)"}

    if rank != 0:
        if world > 1:
            dist.destroy_process_group()
        return
    peak, peak_src = _peaks()
    achieved = tb / (tend_avg * 1e-3) / 1e9
    roof = {"kernel": "ocn_compute_tendencies", "bound": "hbm", "achieved": achieved, "peak": peak, "unit": "GB/s",
            "frac": achieved / peak, "frac_of_8TBps_nominal": achieved / 8000.0, "traffic": None, "peak_source": peak_src,
            "algorithmic_bytes_per_launch": tb, "bytes_per_cell": tb / cells, "avg_launch_ms": tend_avg,
            "n_in_fields": n_in, "n_out_fields": n_out, "share_of_step": 3 * tend_avg / (ms / K),
            "note": "compulsory-bytes HBM roofline as the north_star asks; the kernel is FP64-ALU-bound (DESIGN.md 'Roofline')"}
    line = {"metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": K, "warmup": args.warmup,
            "ms_per_step": ms / K, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
            "dtype": cfg["dtype"], "data": "synthetic",
            "config": {"workload": "%s (%s)" % (args.workload, cfg["description"]), "grid": [g["Nx"], g["Ny"], g["Nz"]],
                       "substages_per_step": 3, "dt": dt, "l2": "inputs larger than L2 (no flush)" if big else
                       "working set fits L2: HBM fraction not meaningful", "parallelism": "replicas x%d" % world,
                       "kernel": {0: "auto", 1: "percell", 2: "fused"}[args.kernel], "state_finite_after_run": finite},
            "clocks": clocks, "e2e": e2e, "gpu_launches": launches, "roofline": roof, "breakdown_ms": breakdown}
    if world == 1 and not args.no_cpu_baseline:
        v, cores, sample, sec, _ = cpu_oracle_leg(args.workload)
        line["cpu_baseline"] = {"value": v, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": sample, "seconds": sec}
    print(json.dumps(line), flush=True)
    if world > 1:
        dist.destroy_process_group()


if __name__ == "__main__":
    main()
