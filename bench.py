"""bench.py — tendency+RK3 cell-updates/s of the hot path on the B200 (BASELINE.json metric).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--workload C2] [--impl ours|reference]

One *step* = one full RK3 time step of the workload = 3 substages, each {ocn_fill_halos, [C3: ocn_compute_w,
ocn_compute_phy], ocn_tendencies_rk3 (= ocn_compute_tendencies + ocn_rk3_substage in one pass; --unfused runs the
two calls)} through the C ABI of libocn.so, on seeded synthetic fields resident in HBM.  value = Nx*Ny*Nz*3*K*N / elapsed (cell-updates/s, whole job).  The default workload is
C2 (512x512x256 fp64, the configuration the north_star's roofline target is quoted on; every field is 562 MB,
far larger than the 126 MB L2, so no flush is needed between iterations).

  * `value`    : K steps through the step-level entry point a user calls (ocn_step_fused; ocn_step for the two-pass paths;
                 ocn_step_model with --project / --free-surface) on a non-default stream, so the library replays its CUDA
                 graph of the sequence (include/ocn.h ocn_grid_set_graphs; --no-graph issues the kernels one by one).
  * `e2e`      : the same metric through ocn_step_host (pinned HOST buffers in, HOST buffers out, copies timed).
  * `roofline` : the fused tendency kernel: algorithmic flops per launch / its CUDA-event duration, measured live with
                 events around every tendency launch of K further steps issued call by call on the same stream
                 (`roofline.call_by_call_ms_per_step` is that region's own step time), against the FP64 (FP32 for C4)
                 issue peak MEASURED in the same run by ocn_alu_probe ("bound": "alu"), and, in `roofline.hbm`, the
                 compulsory-bytes figure against the measured HBM copy peak (MEASURED_PEAKS.json).
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
# cpu_baseline: a bounded sample of the same recipe, ~10-30 s of host work for one full RK3 step
CPU_SAMPLE = {"C0": None, "C1": None, "C2": (512, 512, 128), "C3": (1440, 600, 50), "C4": (512, 512, 128)}
# --impl reference: each of the K + W steps is one full RK3 step on this smaller sample (~1 s each on 16 cores)
REF_SAMPLE = {"C0": None, "C1": None, "C2": (256, 256, 64), "C3": (360, 300, 50), "C4": (256, 256, 64)}
SM_COUNT, SM_GHZ = 148, 1.965          # B200: B200_PROFILING.md (148 SMs, clocks.max.sm 1965 MHz)
ALU_PEAK_TFLOPS = {"f64": SM_COUNT * 64 * 2 * SM_GHZ * 1e-3,     # 4 sub-partitions x 16 FP64 lanes, DFMA = 2 flop
                   "f32": SM_COUNT * 128 * 2 * SM_GHZ * 1e-3}    # 4 x 32 FP32 lanes, FFMA = 2 flop


def _peaks():
    try:
        with open(os.path.join(ROOT, "MEASURED_PEAKS.json")) as f:
            p = json.load(f)
        return float(p["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs)"
    except Exception:
        return 6650.0, "fallback (B200_PROFILING.md 6.65 TB/s)"


def measure_alu_peak(B, torch, dtype, modes=(0,), threads=1024, n_iter=4000, reps=5):
    """FP64 / FP32 issue peak of this GPU, measured: ocn_alu_probe (register-resident FMA chains, include/ocn.h) timed with CUDA
    events on the current stream, best of `reps`.  Returns {mode: TFLOP/s}.  (MEASURED_PEAKS.json has no ALU peak.)"""
    code = 0 if dtype == "f64" else 1
    sink = torch.zeros(SM_COUNT * threads, dtype=torch.float64 if code == 0 else torch.float32, device="cuda")
    out = {}
    for mode in modes:
        for _ in range(2):
            B.ocn_alu_probe(code, mode, SM_COUNT, threads, n_iter, sink)
        best = None
        for _ in range(reps):
            a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            a.record()
            fl = B.ocn_alu_probe(code, mode, SM_COUNT, threads, n_iter, sink)
            b.record()
            torch.cuda.synchronize()
            t = a.elapsed_time(b)
            best = t if best is None else min(best, t)
        out[mode] = fl / (best * 1e-3) / 1e12
    return out


ALU_MODES = {0: "pure FMA, 8 chains/thread, 2 uniform operands"}


def alu_peak_report():
    """`bench.py --alu-peak`: the probe's table for both precisions (the log is kept under profiles/)."""
    import torch
    from paper_2502_14148_b200 import binding as B
    B.lib()
    torch.cuda.set_device(0)
    rows = {}
    for dtype in ("f64", "f32"):
        r = measure_alu_peak(B, torch, dtype, modes=tuple(ALU_MODES))
        rows[dtype] = {"mode %d: %s" % (m, ALU_MODES[m]): round(v, 2) for m, v in r.items()}
        cyc = {m: 2.0 * SM_COUNT * (32 * 4) * SM_GHZ * 1e-3 / v for m, v in r.items()}
        rows[dtype + "_cycles_per_warp_instruction_per_scheduler"] = {"mode %d" % m: round(c, 3) for m, c in cyc.items()}
    print(json.dumps({"alu_probe": rows, "unit": "TFLOP/s", "threads_per_sm": 1024, "derived_peak": ALU_PEAK_TFLOPS}), flush=True)


def _ncu_traffic(key):
    """dram__bytes_read.sum + dram__bytes_write.sum per launch of the dominant kernel, from the committed
    `ncu --set full` summaries (profiles/ncu_traffic.csv: key,bytes,source); None when that kernel/workload was not captured."""
    try:
        with open(os.path.join(ROOT, "profiles", "ncu_traffic.csv")) as f:
            for line in f:
                parts = line.strip().split(",")
                if parts[0] == key:
                    return float(parts[1])
    except Exception:
        pass
    return None


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


def algorithmic_work(cfg, padded_elems, fused_rk3, stage23_share):
    """Algorithmic (compulsory) bytes and flops of ONE launch of the tendency kernel.
    bytes: every input field read once over the padded extents, every output field written once over the interior
    (north_star); with the substage fused in, also G_prev read (stages 2, 3) and the new state written.
    flops: adds + multiplies + divides of the formulas as written, each face flux once: 76 per WENO5-Z
    reconstruction, 7 per Centered(4) advecting velocity (3 per Centered(2)), 3 per face flux (product + divergence),
    13 per 7-point Laplacian, 20 for Coriolis + buoyancy / pressure gradient, 3 per prognostic field for (A4)."""
    p, g = cfg["params"], cfg["grid"]
    esz = 8 if cfg["dtype"] == "f64" else 4
    interior = g["Nx"] * g["Ny"] * g["Nz"]
    flat_z = g["topology"][2] == 2
    mom = bool(p["momentum_prognostic"])
    nt = p["n_tracers"]
    n_vel = 2 if flat_z else 3
    n_in = nt + n_vel + (1 if p["hydrostatic"] else 0)
    n_mom = 0 if not mom else (2 if (p["hydrostatic"] or flat_z) else 3)
    n_out = nt + n_mom
    nbytes = esz * (n_in * padded_elems + n_out * interior)
    if fused_rk3:
        nbytes += esz * interior * n_out * (1.0 + stage23_share)       # q_new written; G_prev read at stages 2, 3
    ndir = 2 if flat_z else 3
    weno_dirs = sum(1 for a in ("adv_x", "adv_y", "adv_z")[:ndir] if p[a] in (5, 7, 9))
    other_dirs = ndir - weno_dirs
    fields = nt + n_mom
    order = max([p[a] for a in ("adv_x", "adv_y", "adv_z")[:ndir] if p[a] in (5, 7, 9)] or [5])
    # per reconstruction, as written: 76 (WENO5, (B8)/(B9) + sums-of-squares indicators); WENO7 / WENO9 in the standard
    # value form: r(1.5 r^2 + 3.5 r + 3) + 6r - 2 = 186 / 318; Centered(4/6/8): 7 / 8 / 11
    rec = {5: 76, 7: 186, 9: 318}[order]
    cen = {5: 7, 7: 8, 9: 11}[order]
    flops = fields * (rec * weno_dirs + 2 * other_dirs)                 # reconstructions
    flops += n_mom * (cen * weno_dirs + 3 * other_dirs)                 # advecting velocities (B21)
    flops += fields * ndir * 3                                          # flux product + divergence
    flops += fields * 13                                                # Laplacians
    flops += 20 if mom else 0                                           # Coriolis, buoyancy / pressure gradient
    if fused_rk3:
        flops += 3 * fields
    return nbytes, flops, n_in, n_out


def max_over_ranks(ms, device=None):
    """device-timed milliseconds -> MAX over all ranks (every multi-GPU number is the slowest rank's)."""
    import torch
    import torch.distributed as dist
    if not (dist.is_available() and dist.is_initialized()) or dist.get_world_size() == 1:
        return float(ms)
    t = torch.tensor([ms], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def whole_job_value(cells_per_rank, substages, steps, world, ms):
    """replicas only: every rank advances its own copy of the workload, so the job processed
    world x cells x substages x steps cell-updates in the time of the slowest rank."""
    return cells_per_rank * substages * steps * world / (ms * 1e-3)


def cpu_oracle_leg(name, size, steps=1, warmup=0, weno_order=5):
    """the oracle as it stands (double / float instantiation, OpenMP over the host cores) on a bounded sample of the
    workload: the same recipe on a sub-grid, `steps` full RK3 steps after `warmup` untimed ones.
    Returns (cell-updates/s, cores, sample text, seconds, cfg)."""
    from oracle import ocnref as ref
    from paper_2502_14148_b200 import workloads as W
    cfg = W.get_config(name, size=size, weno_order=weno_order)
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
    oracle, as it stands, timed on the host cores: W untimed + exactly K timed steps, each one full RK3 step on a
    bounded sample of the workload.  Rank 0 only; the other ranks exit without work."""
    if rank != 0:
        return
    steps, warm = max(1, args.steps), max(0, args.warmup)
    v, cores, sample, dt, cfg = cpu_oracle_leg(args.workload, REF_SAMPLE[args.workload], steps=steps, warmup=warm, weno_order=args.weno_order)
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
    ap.add_argument("--unfused", action="store_true",
                    help="ocn_compute_tendencies + ocn_rk3_substage as two passes instead of ocn_tendencies_rk3")
    ap.add_argument("--weno-order", type=int, default=5, choices=[5, 7, 9],
                    help="7 / 9: the SURVEY 8(f) N1 variant of the workload (halo 4 / 5, high-order kernel, two-pass substage)")
    ap.add_argument("--project", action="store_true",
                    help="N2: append the pressure correction (A11),(A12) to every substage (nonhydrostatic workloads); "
                         "the default times the north_star path (tendency + RK3) without it")
    ap.add_argument("--free-surface", action="store_true",
                    help="N4: append the split-explicit free surface (A13)-(A21) to every substage (hydrostatic workload C3)")
    ap.add_argument("--alu-peak", action="store_true", help="print the ocn_alu_probe table (measured FP64 / FP32 issue peaks) and exit")
    ap.add_argument("--shard", default="none", choices=["none", "y"],
                    help="y: ONE grid split into y-slabs over the N ranks (strong scaling; one neighbour halo exchange per substage, "
                         "include/ocn.h ocn_grid_set_external_halo); default: N independent replicas (weak)")
    ap.add_argument("--no-graph", action="store_true", help="disable the library's CUDA-graph replay of the step sequence")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-e2e", action="store_true")
    args = ap.parse_args()
    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if args.impl == "reference":
        return reference_arm(args, rank, world)
    if args.alu_peak:
        return alu_peak_report()
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

    cfg = W.get_config(args.workload, weno_order=args.weno_order)
    p, g = cfg["params"], cfg["grid"]
    hydro = bool(p["hydrostatic"])
    dev = torch.device("cuda", local)
    big = g["Nx"] * g["Ny"] * g["Nz"] > 4_000_000
    state0 = W.generate_state(cfg, device=dev if big else "cpu", as_numpy=False)
    slabs = None
    global_cells = g["Nx"] * g["Ny"] * g["Nz"]
    if args.shard == "y":
        # strong scaling: this rank owns rows j0 .. j0 + ny_local - 1 of the ONE global grid
        from paper_2502_14148_b200.slab import YSlabs
        if g["topology"][1] != 0:
            raise SystemExit("bench.py --shard y: y-slabs need a Periodic y axis (C1, C2, C4)")
        slabs = YSlabs(g["Ny"], g["halo"], world, rank)
        Hh = g["halo"]
        rows = slice(Hh + slabs.j0, Hh + slabs.j0 + slabs.ny_local)

        def cut(a):
            if a is None:
                return None
            z = torch.zeros_like(a[:, :Hh, :])
            return torch.cat([z, a[:, rows, :], z], dim=1).contiguous()
        state0 = {"u": cut(state0["u"]), "v": cut(state0["v"]), "w": cut(state0["w"]), "c": [cut(c) for c in state0["c"]]}
        g = dict(g, Ny=slabs.ny_local)
        cfg = dict(cfg, grid=g)
    grid = B.ocn_grid_create(g["Nx"], g["Ny"], g["Nz"], g["halo"], g["dx"], g["dy"], g["dz_c"], g["dz_uniform"],
                             g["topology"], cfg["dtype"], device=dev)
    grid.set_kernel(args.kernel)
    if slabs is not None:
        grid.set_external_halo(1, True)
    st = grid.fields_from_state(state0)
    del state0
    torch.cuda.empty_cache()
    hasw = g["topology"][2] != 2 and not hydro
    mom = bool(p["momentum_prognostic"])
    mkG = lambda: grid.fields(n_tracers=p["n_tracers"], u=mom, v=mom, w=mom and hasw)
    G, Gp = mkG(), mkG()
    phy = grid.new_field() if hydro else None
    if slabs is not None:
        p = slabs.local_params(p, g["dy"])      # beta-plane Coriolis is evaluated from the local row index
    cp = B.make_params(p)
    dt = cfg["dt"]
    cells = g["Nx"] * g["Ny"] * g["Nz"]
    L = grid.layout
    padded = L.nx_pad * L.ny_pad * L.nz_pad

    # the fused tendency+substage pass needs the fused kernel (C1-C4 physics) and a second set of state buffers
    fused = not args.unfused and args.kernel != 1
    alt = None
    if fused:
        if not mom:          # prescribed velocities (C0): they carry no tendency and are shared by the ping-pong pair
            alt = B.Fields(st.u, st.v, st.w, [grid.new_field() for _ in st.c])
        else:
            alt = B.Fields(grid.new_field(), grid.new_field(), st.w if (hydro or st.w is None) else grid.new_field(),
                           [grid.new_field() for _ in st.c])
        try:
            B.ocn_tendencies_rk3(grid, cp, 1, 0.0, st, phy, G, None, alt)      # dt = 0: a probe that changes nothing
        except B.OcnError as e:
            if e.code != B.OCN_ERR_UNSUPPORTED:
                raise
            fused, alt = False, None
    tb, flops, n_in, n_out = algorithmic_work(cfg, padded, fused, 2.0 / 3.0)
    bufs = {"cur": st, "alt": alt}
    # N2: pressure solver for the nonhydrostatic workloads (Periodic x,y / Bounded z)
    nonhydro3d = mom and hasw and tuple(g["topology"]) == (0, 0, 1) and slabs is None   # the FFT solver is not sharded
    if args.project and not nonhydro3d:
        raise SystemExit("bench.py --project: the pressure correction applies to the nonhydrostatic workloads (C1, C2, C4)")
    poisson = B.ocn_poisson_create(grid) if nonhydro3d else None
    p_nh = grid.new_field() if nonhydro3d else None
    gam_zet = [(8.0 / 15.0, 0.0), (5.0 / 12.0, 17.0 / 60.0), (3.0 / 4.0, 5.0 / 12.0)]
    # N4: split-explicit free surface for the hydrostatic workload; 30 barotropic substeps per substage interval
    if args.free_surface and not (hydro and mom):
        raise SystemExit("bench.py --free-surface: the split-explicit free surface applies to the hydrostatic workload (C3)")
    bt = B.Barotropic(grid) if (hydro and mom) else None
    bt_N = 30
    bt_w = W.barotropic_weights(bt_N)
    if bt is not None:
        B.ocn_barotropic_init(grid, st, bt)

    xbufs = slabs.make_buffers(B, grid, cp) if slabs is not None else None

    def substage(m, Gm, Gq, ev=None):
        cur = bufs["cur"]
        B.ocn_fill_halos(grid, cp, cur)
        if slabs is not None:       # the one exchange step of the path: H rows of every field to each y-neighbour
            slabs.exchange(B, grid, cp, cur, xbufs)
        if hydro:
            B.ocn_compute_w(grid, cur)
            B.ocn_compute_phy(grid, cp, cur, phy)
        if ev is not None:
            ev[0].record()
        if fused:
            B.ocn_tendencies_rk3(grid, cp, m, dt, cur, phy, Gm, None if m == 1 else Gq, bufs["alt"])
            bufs["cur"], bufs["alt"] = bufs["alt"], cur
        else:
            B.ocn_compute_tendencies(grid, cp, cur, phy, Gm)
        if ev is not None:
            ev[1].record()
        if not fused:
            B.ocn_rk3_substage(grid, cp, m, dt, cur, Gm, None if m == 1 else Gq)
        if args.free_surface:
            gz = gam_zet[m - 1]
            B.ocn_barotropic_forcing(grid, gz[0] / (gz[0] - gz[1]), gz[1] / (gz[0] - gz[1]), Gm, None if m == 1 else Gq, bt)
            B.ocn_barotropic_substeps(grid, p["g"], dt * (gz[0] - gz[1]), bt_N, bt_w, bt)
            B.ocn_barotropic_correct(grid, bufs["cur"], bt)
        if args.project:
            B.ocn_pressure_correction(poisson, dt * (gam_zet[m - 1][0] - gam_zet[m - 1][1]), bufs["cur"], p_nh)

    def step(evs=None):
        a, b = G, Gp
        for m in (1, 2, 3):
            substage(m, a, b, None if evs is None else evs[m - 1])
            a, b = b, a

    # the step-level entry point a user calls: the library replays its CUDA graph of the sequence on a non-default stream
    model_kw = {}
    if args.project:
        model_kw = dict(poisson=poisson, p_nh=p_nh)
    if args.free_surface:
        model_kw = dict(bt=bt, bt_N=bt_N, bt_weights=bt_w)
    if slabs is not None:
        api_name = "call by call: fill_halos, y-slab exchange (torch.distributed P2P), tendencies_rk3"
        api_step = step
    elif model_kw and not fused:
        api_name = "call by call (ocn_step_model needs the fused kernel)"
        api_step = step
    elif model_kw:
        api_name = "ocn_step_model"

        def api_step():
            cur = bufs["cur"]
            B.ocn_step_model(grid, cp, 3, dt, cur, bufs["alt"], G, Gp, p_hy=phy, **model_kw)
            bufs["cur"], bufs["alt"] = bufs["alt"], cur
    elif fused:
        api_name = "ocn_step_fused"

        def api_step():
            cur = bufs["cur"]
            B.ocn_step_fused(grid, cp, 3, dt, cur, bufs["alt"], G, Gp, phy)
            bufs["cur"], bufs["alt"] = bufs["alt"], cur
    else:
        api_name = "ocn_step"

        def api_step():
            B.ocn_step(grid, cp, 3, dt, bufs["cur"], G, Gp, phy)

    def sync():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    grid.set_graphs(not args.no_graph)
    torch.cuda.synchronize()
    torch.cuda.set_stream(torch.cuda.Stream(device=dev))      # CUDA graphs cannot be captured on the legacy default stream
    for _ in range(args.warmup):
        api_step()
    # the library builds a CUDA graph per call sequence on the sequence's SECOND call, and the ping-pong entry points alternate between
    # two sequences (state <-> state_alt): keep warming up (untimed, at most 4 more steps) until two consecutive steps were graph replays,
    # so that no graph instantiation lands in the timed region (it is 100s of microseconds of host work: visible only on C0 / C1)
    priming = 0
    if not args.no_graph and slabs is None:
        streak = 0
        while streak < 2 and priming < 4:
            rb = grid.graph_replays()
            api_step()
            priming += 1
            streak = streak + 1 if grid.graph_replays() > rb else 0
    K = args.steps
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    sampler = ClockSampler(local)
    sampler.start()
    sync()
    n0 = B.ocn_launch_count()
    r0 = grid.graph_replays()
    e0.record()
    for k in range(K):
        api_step()
    e1.record()
    sync()
    launches = B.ocn_launch_count() - n0
    replays = grid.graph_replays() - r0
    ms = e0.elapsed_time(e1)
    ms = max_over_ranks(ms, dev)
    value = whole_job_value(cells, 3, K, world, ms) if slabs is None else global_cells * 3 * K / (ms * 1e-3)
    # ---- the same K steps issued call by call with CUDA events around every tendency launch (roofline instrumentation)
    evs = [[(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(3)] for _ in range(K)]
    c0, c1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    step()
    sync()
    c0.record()
    for k in range(K):
        step(evs[k])
    c1.record()
    sync()
    clocks = sampler.stop()
    cbc_ms = c0.elapsed_time(c1) / K
    tend_ms = [a.elapsed_time(b) for row in evs for (a, b) in row]
    tend_avg = sum(tend_ms) / len(tend_ms)
    st = bufs["cur"]
    finite = all(bool(torch.isfinite(t).all()) for t in st.all())

    # ---- per-call breakdown (diagnostic pass after the timed region; not part of `value`)
    def timed(fn, n=10, warm=3):
        a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        for _ in range(warm):
            fn()
        torch.cuda.synchronize(); a.record()
        for _ in range(n):
            fn()
        b.record(); torch.cuda.synchronize()
        return a.elapsed_time(b) / n
    breakdown = {"fill_halos": timed(lambda: B.ocn_fill_halos(grid, cp, st)),
                 ("tendencies_rk3_fused" if fused else "tendencies"): tend_avg,
                 "rk3_substage_stage1_standalone": timed(lambda: B.ocn_substage(grid, cp, 0.0, 0.0, dt, st, G, None)),
                 "rk3_substage_stage23_standalone": timed(lambda: B.ocn_substage(grid, cp, 0.0, 1e-300, dt, st, G, Gp))}
    if fused:
        breakdown["tendencies_only"] = timed(lambda: B.ocn_compute_tendencies(grid, cp, st, phy, G))
    if nonhydro3d:      # N2, timed call by call on the final state (diagnostic; the correction is idempotent up to rounding)
        breakdown["n2_pressure_rhs"] = timed(lambda: B.ocn_pressure_rhs(grid, dt, st, p_nh))
        breakdown["n2_poisson_solve"] = timed(lambda: B.ocn_poisson_solve(poisson, p_nh, p_nh))
        B.ocn_pressure_rhs(grid, dt, st, p_nh)
        B.ocn_poisson_solve(poisson, p_nh, p_nh)
        breakdown["n2_pressure_correct"] = timed(lambda: B.ocn_pressure_correct(grid, dt, st, p_nh))
        breakdown["n2_pressure_correction_total"] = timed(lambda: B.ocn_pressure_correction(poisson, dt, st, p_nh))
    if g["topology"][2] == 1:      # N3: one implicit vertical solve of every prognostic field (diagnostic, stage-1 interval)
        breakdown["n3_implicit_vertical_diffusion"] = timed(lambda: B.ocn_implicit_vertical_diffusion(grid, cp, dt * 8.0 / 15.0, st))
    if bt is not None:      # N4, call by call (diagnostic)
        breakdown["n4_barotropic_forcing"] = timed(lambda: B.ocn_barotropic_forcing(grid, 1.5, 0.5, G, Gp, bt))
        breakdown["n4_barotropic_substeps_N%d_M%d" % (bt_N, len(bt_w))] = timed(lambda: B.ocn_barotropic_substeps(grid, p["g"], dt, bt_N, bt_w, bt))
        breakdown["n4_barotropic_correct"] = timed(lambda: B.ocn_barotropic_correct(grid, st, bt))
    if hydro:
        breakdown["compute_w"] = timed(lambda: B.ocn_compute_w(grid, st))
        breakdown["compute_phy"] = timed(lambda: B.ocn_compute_phy(grid, cp, st, phy))

    # ---- end to end: HOST buffers in, HOST buffers out, through ocn_step_host
    e2e = None
    if not args.no_e2e and slabs is None:
        host = B.Fields(*[None if t is None else torch.empty_like(t, device="cpu").pin_memory() for t in (st.u, st.v, st.w)],
                        [torch.empty_like(t, device="cpu").pin_memory() for t in st.c])
        for h, d in zip(host.all(), st.all()):
            h.copy_(d)
        esz = 8 if cfg["dtype"] == "f64" else 4
        nf_in = len(host.all())
        nf_out = (p["n_tracers"] + ((3 if hasw else 2) if mom else 0))
        Ke = max(1, min(K, 3))
        other = bufs["alt"] if fused else None
        B.ocn_step_host(grid, cp, 3, dt, host, st, other, G, Gp, phy)      # warm-up
        sync()
        a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        a.record()
        for _ in range(Ke):
            B.ocn_step_host(grid, cp, 3, dt, host, st, other, G, Gp, phy)
        b.record()
        sync()
        ems = a.elapsed_time(b)
        ems = max_over_ranks(ems, dev)
        e2e = {"value": whole_job_value(cells, 3, Ke, world, ems), "unit": UNIT, "h2d_bytes_per_step": nf_in * L.n_alloc * esz,
               "d2h_bytes_per_step": nf_out * L.n_alloc * esz, "steps": Ke, "ms_per_step": ems / Ke,
               "api": "ocn_step_host (pinned host buffers; all state fields in, all prognostic fields out, every step)"}

    if rank != 0:
        if world > 1:
            dist.destroy_process_group()
        return
    hbm_peak, hbm_src = _peaks()
    alu_derived = ALU_PEAK_TFLOPS[cfg["dtype"]]
    alu_peak = measure_alu_peak(B, torch, cfg["dtype"])[0]
    kname = ("ocn_tendencies_rk3 (tend_hiorder_tma_kernel, WENO%d, substage fused)" % args.weno_order if fused and args.weno_order != 5 else
             "ocn_tendencies_rk3 (tend_percell_kernel, substage fused)" if fused and (args.kernel == 1 or args.workload == "C0") else
             "ocn_tendencies_rk3 (tend_fused_kernel, FUSE_RK3)" if fused else
             "ocn_compute_tendencies (tend_hiorder kernels, WENO%d)" % args.weno_order if args.weno_order != 5 else
             "ocn_compute_tendencies (%s)" % ("tend_percell_kernel" if args.kernel == 1 or not big and args.workload == "C0"
                                              else "tend_fused_kernel where it applies"))
    tflops = flops * cells / (tend_avg * 1e-3) / 1e12
    gbs = tb / (tend_avg * 1e-3) / 1e9
    traffic = _ncu_traffic("%s%s:%s" % (args.workload, "" if args.weno_order == 5 else "-weno%d" % args.weno_order,
                                        "fused_rk3" if fused else "tendencies"))
    roof = {"kernel": kname, "bound": "alu", "achieved": tflops, "peak": alu_peak, "unit": "TFLOP/s", "frac": tflops / alu_peak,
            "traffic": traffic,
            "peak_source": "measured in this run: ocn_alu_probe mode 0 (register-resident %s chains, 148 blocks x 1024 threads, best "
                           "of 5, CUDA events); derived figure 148 SMs x %d lanes x 2 flop x 1.965 GHz = %.2f" % (
                               "DFMA" if cfg["dtype"] == "f64" else "FFMA", 64 if cfg["dtype"] == "f64" else 128, alu_derived),
            "peak_derived": alu_derived,
            "algorithmic_flops_per_cell": flops, "algorithmic_flops_per_launch": flops * cells, "avg_launch_ms": tend_avg,
            "share_of_step": 3 * tend_avg / cbc_ms, "call_by_call_ms_per_step": cbc_ms,
            "hbm": {"achieved": gbs, "peak": hbm_peak, "unit": "GB/s", "frac": gbs / hbm_peak,
                    "frac_of_8TBps_nominal": gbs / 8000.0, "peak_source": hbm_src, "algorithmic_bytes_per_launch": tb,
                    "bytes_per_cell": tb / cells, "n_in_fields": n_in, "n_out_fields": n_out,
                    "note": "compulsory-bytes HBM roofline the north_star asks for; this kernel is bound by the FP64 "
                            "issue rate, not HBM (DESIGN.md 6)"}}
    # HBM rooflines of the N2 / N3 / N4 calls from the diagnostic pass (algorithmic bytes per call:
    # every field a call must read once + every field it must write once, interior cells)
    esz = 8 if cfg["dtype"] == "f64" else 4
    fld = cells * esz
    next_rows = {}

    def hbm_row(key, ms_, nbytes, what):
        next_rows[key] = {"ms": ms_, "algorithmic_bytes": nbytes, "achieved": nbytes / (ms_ * 1e-3) / 1e9, "peak": hbm_peak,
                          "unit": "GB/s", "frac": nbytes / (ms_ * 1e-3) / 1e9 / hbm_peak, "bytes": what}
    if "n2_pressure_correction_total" in breakdown:
        hbm_row("n2_pressure_rhs", breakdown["n2_pressure_rhs"], 4 * fld, "u,v,w read + rhs written")
        hbm_row("n2_poisson_solve", breakdown["n2_poisson_solve"], 10 * fld, "2 x (x-FFT + y-FFT: read + write each) + Thomas read + write")
        hbm_row("n2_pressure_correct", breakdown["n2_pressure_correct"], 7 * fld, "p,u,v,w read + u,v,w written")
    if "n3_implicit_vertical_diffusion" in breakdown:
        nprog = (2 if mom else 0) + (1 if (mom and hasw) else 0) + p["n_tracers"]
        hbm_row("n3_implicit_vertical_diffusion", breakdown["n3_implicit_vertical_diffusion"], 2 * nprog * fld, "%d fields read + written" % nprog)
    if "n4_barotropic_correct" in breakdown:
        hbm_row("n4_barotropic_forcing", breakdown["n4_barotropic_forcing"], 4 * fld, "G_u, G_v, G_prev_u, G_prev_v read")
        hbm_row("n4_barotropic_correct", breakdown["n4_barotropic_correct"], 4 * fld, "u,v read + written")
    line = {"metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": K, "warmup": args.warmup,
            "ms_per_step": ms / K, "higher_is_better": True, "scaling": "weak" if slabs is None else "strong", "vs_baseline": None,
            "dtype": cfg["dtype"], "data": "synthetic",
            "config": {"workload": "%s (%s)" % (args.workload, cfg["description"]), "grid": [g["Nx"], g["Ny"], g["Nz"]],
                       "substages_per_step": 3, "dt": dt, "l2": "inputs larger than L2 (no flush)" if big else
                       "working set fits L2: HBM fraction not meaningful", "parallelism": ("replicas x%d" % world) if slabs is None else
                       "y-slabs x%d of the one %dx%dx%d grid, neighbour halo exchange of %d rows per side per substage" % (
                           world, g["Nx"], slabs.Ny, g["Nz"], g["halo"]),
                       "kernel": {0: "auto", 1: "percell", 2: "fused"}[args.kernel],
                       "substage_path": "fill_halos + " + ("" if not hydro else "p_hy scan + " if (fused and slabs is None and args.kernel != 1
                                                                                                     and args.weno_order == 5)
                                                            else "w, p_hy scans + ")
                                        + ("tendencies_rk3 (one pass, ping-pong state%s)" % (
                                            "; w diagnosed inside the kernel" if hydro and slabs is None and args.kernel != 1 and args.weno_order == 5 else "")
                                           if fused else "compute_tendencies + rk3_substage")
                                        + (" + pressure_correction (N2: rhs, cuFFT + Thomas solve, correct)" if args.project else "")
                                        + (" + split-explicit free surface (N4: forcing, %d substeps, correct)" % len(bt_w) if args.free_surface else ""),
                       "entry_point": api_name, "cuda_graph": (not args.no_graph), "graph_replays_in_timed_region": replays,
                       "untimed_graph_priming_steps_after_warmup": priming,
                       "state_finite_after_run": finite},
            "clocks": clocks, "e2e": e2e, "gpu_launches": launches, "roofline": roof, "breakdown_ms": breakdown,
            "next_rows_hbm": next_rows}
    if world == 1 and not args.no_cpu_baseline:
        smp = CPU_SAMPLE[args.workload]
        if smp is not None and args.weno_order != 5:
            smp = (smp[0] // 2, smp[1] // 2, smp[2])       # the general WENO7/9 oracle routine is ~4x slower per cell
        v, cores, sample, sec, _ = cpu_oracle_leg(args.workload, smp, weno_order=args.weno_order)
        line["cpu_baseline"] = {"value": v, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": sample, "seconds": sec}
        # "... on all host cores and on 1 thread": the same oracle on a sample 1/8 the size, one OpenMP thread
        from oracle import ocnref as _ref
        smp1 = None if smp is None else (max(16, smp[0] // 4), max(16, smp[1] // 2), smp[2])
        nthr = _ref.num_threads()
        _ref.set_num_threads(1)
        try:
            v1, _, sample1, sec1, _ = cpu_oracle_leg(args.workload, smp1, weno_order=args.weno_order)
        finally:
            _ref.set_num_threads(nthr)
        line["cpu_baseline"]["one_thread"] = {"value": v1, "unit": UNIT, "cores": 1, "sample": sample1, "seconds": sec1}
    print(json.dumps(line), flush=True)
    if world > 1:
        dist.destroy_process_group()


if __name__ == "__main__":
    main()
