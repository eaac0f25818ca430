"""GPU parity: every call of the hot path, through the C ABI (ctypes binding), against the CPU oracle on the
same seeded inputs (protocol P1 "teacher-forced" per call, P2 chained state after a full step; DESIGN.md
"Parity protocol").  Tolerances are the north_star's: relative max-norm 1e-12 (fp64), 2e-5 (fp32); halo fill
(pure copies) is bitwise.  Run with `pytest -m gpu` on the B200 box."""
import numpy as np
import pytest

from tests import parity_util as PU

pytestmark = pytest.mark.gpu

P, B, F = 0, 1, 2


@pytest.fixture(scope="module")
def binding():
    import torch
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    from paper_2502_14148_b200 import binding as Bd
    Bd.lib()      # raises when libocn.so is missing: no fallback
    return Bd


@pytest.fixture(scope="module")
def W():
    from paper_2502_14148_b200 import workloads
    return workloads


KERNELS = [1, 0]   # OCN_KERNEL_PERCELL, OCN_KERNEL_AUTO (fused where it applies)


def _three_substages(binding, ref, cfg, state, kernel):
    """teacher-forced parity of the three substages of one step; each substage starts from the GPU's state."""
    prev = None
    for stage in (1, 2, 3):
        errs, new_gpu, (Gf, G64), gg = PU.run_substage_parity(binding, ref, cfg, state, kernel=kernel, stage=stage,
                                                              G_prev_pair=prev)
        PU.assert_errs(errs, cfg["dtype"], "%s stage %d kernel %d" % (cfg["name"], stage, kernel))
        prev = (Gf, G64)      # device tendencies (same layout on every Grid of this config) + their float64 copy
        state = new_gpu
    return state


# ------------------------------------------------------------------------------------------ configs
@pytest.mark.parametrize("kernel", KERNELS)
def test_c0_full(binding, ref, W, kernel):
    cfg = W.get_config("C0")
    _three_substages(binding, ref, cfg, W.generate_state(cfg), kernel)


@pytest.mark.parametrize("kernel", KERNELS)
@pytest.mark.parametrize("size", [(40, 24, 20), (67, 35, 9)])
def test_c1_small(binding, ref, W, kernel, size):
    cfg = W.get_config("C1", size=size)
    _three_substages(binding, ref, cfg, W.generate_state(cfg), kernel)


@pytest.mark.parametrize("kernel", KERNELS)
def test_c1_full(binding, ref, W, kernel):
    cfg = W.get_config("C1")
    errs, *_ = PU.run_substage_parity(binding, ref, cfg, W.generate_state(cfg), kernel=kernel, stage=1)
    PU.assert_errs(errs, "f64", "C1 full kernel %d" % kernel)


@pytest.mark.parametrize("kernel", KERNELS)
@pytest.mark.parametrize("size", [(48, 40, 12), (71, 33, 50)])
def test_c3_small(binding, ref, W, kernel, size):
    cfg = W.get_config("C3", size=size)
    _three_substages(binding, ref, cfg, W.generate_state(cfg), kernel)


@pytest.mark.parametrize("kernel", KERNELS)
@pytest.mark.parametrize("size", [(40, 24, 20), (133, 37, 11)])
def test_c4_small_fp32(binding, ref, W, kernel, size):
    cfg = W.get_config("C4", size=size)
    _three_substages(binding, ref, cfg, W.generate_state(cfg), kernel)


@pytest.mark.parametrize("kernel", KERNELS)
def test_c2_physics_with_spectrum_small(binding, ref, W, kernel):
    cfg = W.get_config("C2", size=(64, 48, 32))
    _three_substages(binding, ref, cfg, W.generate_state(cfg), kernel)


# ------------------------------------------------------------------------------ chained full step (P2)
@pytest.mark.parametrize("name,size", [("C0", None), ("C1", (40, 24, 20)), ("C3", (48, 40, 12)), ("C4", (40, 24, 20))])
def test_chained_step_state(binding, ref, W, name, size):
    """ocn_step (3 substages, device-resident) against the oracle's chained step: compare the STATE only (H3)."""
    import torch
    cfg = W.get_config(name, size=size)
    p = cfg["params"]
    state = W.generate_state(cfg)
    rg = PU.ref_grid(ref, cfg)
    gg = PU.gpu_grid(binding, cfg)
    st = gg.fields_from_state(state)
    G, Gp = PU.new_G(binding, gg, cfg), PU.new_G(binding, gg, cfg)
    phy = gg.new_field() if p["hydrostatic"] else None
    binding.ocn_step(gg, p, 3, cfg["dt"], st, G, Gp, phy)
    torch.cuda.synchronize()
    got = gg.state_from_fields(st)
    want = PU.to64(state)
    ref.step(rg, p, 3, cfg["dt"], want, eval=0)
    tol = {"f64": 1e-12, "f32": 2e-5}[cfg["dtype"]]
    for (nm, a), (_, b) in zip(PU.named(got), PU.named(want)):
        if nm == "w" and p["hydrostatic"]:
            continue
        e, den = PU.rel_err(rg, a, b)
        assert e <= tol, "%s chained state %s: %g" % (name, nm, e)


def test_step_host_matches_step(binding, ref, W):
    """the end-to-end entry point (host buffers in, host buffers out) gives bit-identical state to ocn_step."""
    import torch
    cfg = W.get_config("C1", size=(40, 24, 20))
    p = cfg["params"]
    state = W.generate_state(cfg)
    gg = PU.gpu_grid(binding, cfg)
    st = gg.fields_from_state(state)
    G, Gp = PU.new_G(binding, gg, cfg), PU.new_G(binding, gg, cfg)
    binding.ocn_step(gg, p, 3, cfg["dt"], st, G, Gp, None)
    torch.cuda.synchronize()
    want = gg.state_from_fields(st)
    dev = gg.fields_from_state(state)
    host = binding.Fields(*[t.cpu().pin_memory() for t in (dev.u, dev.v, dev.w)], [t.cpu().pin_memory() for t in dev.c])
    dev2 = gg.fields(n_tracers=p["n_tracers"])
    binding.ocn_step_host(gg, p, 3, cfg["dt"], host, dev2, G, Gp, None)
    torch.cuda.synchronize()
    L = gg.layout
    for nm, t in (("u", host.u), ("v", host.v), ("w", host.w), ("c0", host.c[0]), ("c1", host.c[1])):
        a = t.view(L.nz_pad, L.ny_pad, L.stride_y)[:, :, gg._xo:gg._xo + L.nx_pad].numpy()
        b = want[nm] if nm in want else want["c"][int(nm[1:])]
        assert np.array_equal(PU.ref_grid(ref, cfg).interior(a), PU.ref_grid(ref, cfg).interior(b)), nm
