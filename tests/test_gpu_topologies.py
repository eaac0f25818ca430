"""GPU parity over every per-axis topology ocn_grid_create accepts (north_star: "per-axis Periodic/Bounded topology"; the paper's
own grids: listing 15 `topology=(Bounded, Flat, Flat)` PAPER.md:940, the LES `RectilinearGrid(... topology ...)` PAPER.md:392-395),
not only the five workloads' (P,P,Flat), (P,P,B), (P,B,B).

The workloads never put a wall in x, never make z periodic and never flatten y, but the default dispatch sends such grids to the same
hand-synchronised kernels: the wall-normal zeroing of the x-strips in the halo fill, the wall face of u in the TMA-ring and marching
kernels (first face of the x loop, the mirrored stencils next to it), the ring planes a periodic-z grid takes from its z-halo, the
substage's skipped wall faces.  Protocol as everywhere (tests/parity_util.run_substage_parity): three substages, teacher-forced, halo
fill bitwise, G and the new state element by element against the oracle, tolerances 1e-12 / 2e-5, plus the increment check.

Physics: the LES terms of C1 (WENO on every non-Flat axis, f-plane Coriolis, buoyancy, Laplacians) on a uniform grid, and the
hydrostatic terms of C3 (stretched z, Centered2 in z, beta-plane, p_hy) for the topologies with Bounded z.  Fields: seeded normal
noise (velocities 0.01, T = 20 + 0.05 n, S = 35 + 0.05 n) — nothing smooth for an index error to hide behind."""
import numpy as np
import pytest

from tests import parity_util as PU

pytestmark = pytest.mark.gpu

P, B_, F = 0, 1, 2
TOPOLOGIES = [(B_, P, B_), (B_, B_, B_), (P, P, P), (P, B_, P), (B_, B_, P), (P, F, B_), (B_, F, F), (F, P, B_)]
SIZE = (37, 22, 11)          # ragged against the 31 x 6 tiles of the TMA-ring kernel and the 32-wide tiles of the marching kernel


@pytest.fixture(scope="module")
def binding():
    import torch
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    from paper_2502_14148_b200 import binding as Bd
    Bd.lib()
    return Bd


def _config(W, base, topology, order, dtype):
    n = [1 if t == F else s for s, t in zip(SIZE, topology)]
    cfg = W.get_config(base, size=tuple(n), weno_order=order)
    cfg = dict(cfg, dtype=dtype, grid=dict(cfg["grid"], topology=tuple(topology)))
    return cfg


def _noise_state(cfg, seed):
    g = cfg["grid"]
    Hh = g["halo"]
    h = [0 if t == F else Hh for t in g["topology"]]
    shape = (g["Nz"] + 2 * h[2], g["Ny"] + 2 * h[1], g["Nx"] + 2 * h[0])
    npdt = np.float64 if cfg["dtype"] == "f64" else np.float32
    r = np.random.default_rng(seed)

    def field(mean, amp):
        a = np.zeros(shape, dtype=npdt)                     # halos left at zero: the fill under test writes them
        a[h[2]:h[2] + g["Nz"], h[1]:h[1] + g["Ny"], h[0]:h[0] + g["Nx"]] = (mean + amp * r.standard_normal((g["Nz"], g["Ny"], g["Nx"]))).astype(npdt)
        return a
    # the velocity component along a Flat axis does not exist
    t = g["topology"]
    state = {"u": field(0.0, 0.01) if t[0] != F else None, "v": field(0.0, 0.01) if t[1] != F else None,
             "w": field(0.0, 0.01) if t[2] != F else None, "c": [field(20.0, 0.05), field(35.0, 0.05)]}
    return state


def _three_substages(binding, ref, cfg, state, kernel, what):
    prev = None
    for stage in (1, 2, 3):
        errs, new_gpu, (Gf, G64), gg = PU.run_substage_parity(binding, ref, cfg, state, kernel=kernel, stage=stage, G_prev_pair=prev)
        PU.assert_errs(errs, cfg["dtype"], "%s stage %d" % (what, stage))
        prev = (Gf, G64)
        state = new_gpu


@pytest.mark.parametrize("dtype", ["f64", "f32"])
@pytest.mark.parametrize("order", [5, 9])
@pytest.mark.parametrize("kernel", [1, 0])                 # OCN_KERNEL_PERCELL, OCN_KERNEL_AUTO (TMA-ring / marching kernels where they apply)
@pytest.mark.parametrize("topology", TOPOLOGIES)
def test_les_physics_on_every_topology(binding, ref, topology, kernel, order, dtype):
    from paper_2502_14148_b200 import workloads as W
    cfg = _config(W, "C1", topology, order, dtype)
    _three_substages(binding, ref, cfg, _noise_state(cfg, 100 + 7 * order + kernel), kernel,
                     "LES %s WENO%d %s kernel %d" % (topology, order, dtype, kernel))


@pytest.mark.parametrize("order", [5, 9])
@pytest.mark.parametrize("kernel", [1, 0])
@pytest.mark.parametrize("topology", [(B_, B_, B_), (B_, P, B_), (P, P, B_), (P, F, B_)])
def test_hydrostatic_physics_with_walls_in_x(binding, ref, topology, kernel, order):
    """C3's terms (w from continuity, p_hy, -grad_h p_hy, beta-plane Coriolis, stretched z) on basins and channels the workload does
    not have; kernel 0 is the hydrostatic TMA-ring instantiation (WENO5) / the marching kernel (WENO9) wherever they apply."""
    from paper_2502_14148_b200 import workloads as W
    cfg = _config(W, "C3", topology, order, "f64")
    _three_substages(binding, ref, cfg, _noise_state(cfg, 300 + order + kernel), kernel, "hydrostatic %s WENO%d kernel %d" % (topology, order, kernel))


@pytest.mark.parametrize("topology", [(B_, P, B_), (B_, B_, B_), (P, P, P), (B_, B_, P)])
@pytest.mark.parametrize("order", [5, 9])
def test_fused_substage_is_bit_identical_to_the_two_calls_on_every_topology(binding, topology, order):
    """ocn_step_fused (tendency + (A4) in one pass; what the bench times) == ocn_step (two kernels, the path compared with the oracle
    above), bit for bit, on the 3-D topologies no workload has."""
    import torch
    from paper_2502_14148_b200 import workloads as W
    B = binding
    cfg = _config(W, "C1", topology, order, "f64")
    p = cfg["params"]
    gg = PU.gpu_grid(B, cfg)
    state = _noise_state(cfg, 500 + order)
    a, b = gg.fields_from_state(state), gg.fields_from_state(state)
    b2 = gg.fields(n_tracers=2)
    Ga, Gpa, Gb, Gpb = (PU.new_G(B, gg, cfg) for _ in range(4))
    B.ocn_step(gg, p, 3, cfg["dt"], a, Ga, Gpa, None)
    B.ocn_step_fused(gg, p, 3, cfg["dt"], b, b2, Gb, Gpb, None)
    torch.cuda.synchronize()
    for nm, x, y in (("u", a.u, b2.u), ("v", a.v, b2.v), ("w", a.w, b2.w), ("T", a.c[0], b2.c[0]), ("S", a.c[1], b2.c[1])):
        assert torch.equal(gg.interior(x), gg.interior(y)), "%s WENO%d: %s differs between ocn_step and ocn_step_fused" % (topology, order, nm)
        assert bool(torch.isfinite(gg.interior(y)).all())
