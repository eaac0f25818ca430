"""GPU parity of the WENO7 / WENO9 path: ocn_fill_halos (halo 4, 5), ocn_compute_tendencies through the
general high-order kernel (tend_hiorder.cu), ocn_rk3_substage — teacher-forced against the long-double oracle, same
tolerances as the WENO5 path (1e-12 fp64, 2e-5 fp32; halo fill bitwise).  Run with `pytest -m gpu` on the B200 box."""
import numpy as np
import pytest

from tests import parity_util as PU

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def binding():
    import torch
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    from paper_2502_14148_b200 import binding as Bd
    Bd.lib()
    return Bd


@pytest.fixture(scope="module")
def W():
    from paper_2502_14148_b200 import workloads
    return workloads


def _three_substages(binding, ref, cfg, state, kernel=0):
    """kernel 0: the marching kernel on 3-D grids (every face flux once); kernel 1: the per-cell high-order kernel"""
    prev = None
    for stage in (1, 2, 3):
        errs, new_gpu, (Gf, G64), gg = PU.run_substage_parity(binding, ref, cfg, state, kernel=kernel, stage=stage, G_prev_pair=prev)
        PU.assert_errs(errs, cfg["dtype"], "%s WENO%d stage %d" % (cfg["name"], cfg["weno_order"], stage))
        prev = (Gf, G64)
        state = new_gpu
    return state


@pytest.mark.parametrize("order", [7, 9])
def test_c0_weno79(binding, ref, W, order):
    cfg = W.get_config("C0", weno_order=order)
    _three_substages(binding, ref, cfg, W.generate_state(cfg))


@pytest.mark.parametrize("kernel", [0, 1])
@pytest.mark.parametrize("order", [7, 9])
@pytest.mark.parametrize("size", [(40, 24, 20), (67, 35, 9)])
def test_c1_weno79(binding, ref, W, order, size, kernel):
    cfg = W.get_config("C1", size=size, weno_order=order)
    _three_substages(binding, ref, cfg, W.generate_state(cfg), kernel)


@pytest.mark.parametrize("order", [7, 9])
def test_c2_spectrum_weno79(binding, ref, W, order):
    cfg = W.get_config("C2", size=(64, 48, 32), weno_order=order)
    _three_substages(binding, ref, cfg, W.generate_state(cfg))


@pytest.mark.parametrize("kernel", [0, 1])
@pytest.mark.parametrize("order", [7, 9])
@pytest.mark.parametrize("size", [(48, 40, 12), (71, 33, 50)])
def test_c3_hydrostatic_weno79(binding, ref, W, order, size, kernel):
    cfg = W.get_config("C3", size=size, weno_order=order)
    _three_substages(binding, ref, cfg, W.generate_state(cfg), kernel)


@pytest.mark.parametrize("kernel", [0, 1])
@pytest.mark.parametrize("order", [7, 9])
def test_c4_fp32_weno79(binding, ref, W, order, kernel):
    cfg = W.get_config("C4", size=(40, 24, 20), weno_order=order)
    _three_substages(binding, ref, cfg, W.generate_state(cfg), kernel)


@pytest.mark.parametrize("order", [7, 9])
@pytest.mark.parametrize("name,size", [("C1", (67, 35, 9)), ("C3", (48, 40, 12)), ("C4", (40, 24, 20))])
def test_unstaged_march_kernel_weno79(binding, ref, W, name, size, order):
    """The global-load marching kernel (the fallback of the TMA-staged one: more than 3 tracers, tiles that do not fit two
    blocks per SM) stays under test through the grid's diagnostic flag OCN_DIAG_HI_NOSTAGE."""
    cfg = dict(W.get_config(name, size=size, weno_order=order), diag=binding.OCN_DIAG_HI_NOSTAGE)
    _three_substages(binding, ref, cfg, W.generate_state(cfg))


@pytest.mark.parametrize("order", [7, 9])
@pytest.mark.parametrize("variant", ["prescribed_velocities", "fp64_three_tracers"])
def test_marching_kernels_off_the_benched_configurations(binding, ref, W, order, variant):
    """The marching kernels on models no workload has: (a) prescribed velocities on a 3-D grid (no momentum tendency: only the
    tracers carry one, the top-edge rows of the staged kernel are taken by rows 0 .. n_tracers-1); (b) three tracers in fp64, whose
    tiles do not fit two blocks per SM at WENO9, so the launcher falls back to the global-load marching kernel by itself."""
    if variant == "prescribed_velocities":
        cfg = W.get_config("C1", size=(67, 35, 9), weno_order=order)
        cfg = dict(cfg, params=dict(cfg["params"], momentum_prognostic=0))
    else:
        cfg = W.get_config("C4", size=(40, 24, 20), weno_order=order)
        cfg = dict(cfg, dtype="f64")
    state = W.generate_state(cfg)
    errs, *_ = PU.run_substage_parity(binding, ref, cfg, state, kernel=0, stage=1)
    PU.assert_errs(errs, cfg["dtype"], "%s WENO%d" % (variant, order))


def _interior_equal(rg, a, b):
    return np.array_equal(rg.interior(np.asarray(a)), rg.interior(np.asarray(b)))


@pytest.mark.parametrize("order", [7, 9])
@pytest.mark.parametrize("name,size,kernel,nostage", [("C1", (40, 24, 20), 0, False), ("C1", (67, 35, 9), 0, False), ("C3", (48, 40, 12), 0, False),
                                                      ("C4", (40, 24, 20), 0, False),
                                                      # the global-load marching kernel and the per-cell kernel (3-D and the 2-D C0)
                                                      ("C1", (67, 35, 9), 0, True), ("C3", (48, 40, 12), 0, True), ("C1", (40, 24, 20), 1, False),
                                                      ("C0", None, 0, False)])
def test_tendencies_rk3_weno79_is_bit_identical_to_the_two_calls(binding, ref, W, name, size, kernel, nostage, order):
    """ocn_tendencies_rk3 on a WENO7/9 model (the (A4) substage fused into the TMA-staged marching kernel, the global-load marching
    kernel or the per-cell kernel; ping-pong state) == ocn_compute_tendencies followed by ocn_rk3_substage, bit for bit, for G and
    for the state, at every stage; the latter sequence is the one checked against the oracle above."""
    import torch
    cfg = W.get_config(name, weno_order=order) if size is None else W.get_config(name, size=size, weno_order=order)
    if nostage:
        cfg = dict(cfg, diag=binding.OCN_DIAG_HI_NOSTAGE)
    p = cfg["params"]
    rg = PU.ref_grid(ref, cfg)
    gg = PU.gpu_grid(binding, cfg, kernel)
    state = W.generate_state(cfg)
    a = gg.fields_from_state(state)                       # path A: separate calls, in place
    b = gg.fields_from_state(state)                       # path B: fused, ping-pong b -> b2 -> b ...
    b2 = gg.fields(n_tracers=p["n_tracers"], w=state.get("w") is not None)
    if not p["momentum_prognostic"]:                      # prescribed velocities are shared by the ping-pong pair
        b2.u, b2.v, b2.w = b.u, b.v, b.w
    Ga, Gpa = PU.new_G(binding, gg, cfg), PU.new_G(binding, gg, cfg)
    Gb, Gpb = PU.new_G(binding, gg, cfg), PU.new_G(binding, gg, cfg)
    phy = gg.new_field() if p["hydrostatic"] else None
    if p["hydrostatic"]:
        b2.w = b.w                                          # the diagnosed w may be shared by the ping-pong pair
    for stage in (1, 2, 3):
        binding.ocn_fill_halos(gg, p, a)
        binding.ocn_fill_halos(gg, p, b)
        if p["hydrostatic"]:
            binding.ocn_compute_w(gg, a); binding.ocn_compute_phy(gg, p, a, phy)
        binding.ocn_compute_tendencies(gg, p, a, phy, Ga)
        binding.ocn_rk3_substage(gg, p, stage, cfg["dt"], a, Ga, None if stage == 1 else Gpa)
        if p["hydrostatic"]:
            binding.ocn_compute_w(gg, b); binding.ocn_compute_phy(gg, p, b, phy)
        binding.ocn_tendencies_rk3(gg, p, stage, cfg["dt"], b, phy, Gb, None if stage == 1 else Gpb, b2)
        torch.cuda.synchronize()
        sa, sb = gg.state_from_fields(a), gg.state_from_fields(b2)
        ga, gb = gg.state_from_fields(Ga), gg.state_from_fields(Gb)
        for (nm, x), (_, y) in zip(PU.named(ga), PU.named(gb)):
            assert _interior_equal(rg, x, y), "%s WENO%d stage %d: G_%s differs" % (name, order, stage, nm)
        for (nm, x), (_, y) in zip(PU.named(sa), PU.named(sb)):
            if nm == "w" and p["hydrostatic"]:
                continue
            assert _interior_equal(rg, x, y), "%s WENO%d stage %d: state %s differs" % (name, order, stage, nm)
        Ga, Gpa = Gpa, Ga
        Gb, Gpb = Gpb, Gb
        b, b2 = b2, b


@pytest.mark.parametrize("order", [7, 9])
def test_step_fused_weno79_matches_step(binding, ref, W, order):
    import torch
    cfg = W.get_config("C1", size=(40, 24, 20), weno_order=order)
    p = cfg["params"]
    rg = PU.ref_grid(ref, cfg)
    gg = PU.gpu_grid(binding, cfg)
    state = W.generate_state(cfg)
    a, b = gg.fields_from_state(state), gg.fields_from_state(state)
    b2 = gg.fields(n_tracers=p["n_tracers"])
    G, Gp = PU.new_G(binding, gg, cfg), PU.new_G(binding, gg, cfg)
    binding.ocn_step(gg, p, 3, cfg["dt"], a, G, Gp, None)
    binding.ocn_step_fused(gg, p, 3, cfg["dt"], b, b2, G, Gp, None)
    torch.cuda.synchronize()
    for (nm, x), (_, y) in zip(PU.named(gg.state_from_fields(a)), PU.named(gg.state_from_fields(b2))):
        assert _interior_equal(rg, x, y), "WENO%d: state %s differs between ocn_step and ocn_step_fused" % (order, nm)


def test_c1_full_weno9(binding, ref, W):
    cfg = W.get_config("C1", weno_order=9)
    errs, *_ = PU.run_substage_parity(binding, ref, cfg, W.generate_state(cfg), kernel=0, stage=1)
    PU.assert_errs(errs, "f64", "C1 full WENO9")


def test_weno79_argument_errors(binding, W):
    """halo < (order+1)/2, mixed orders and forcing the fused kernel are refused before anything is enqueued."""
    cfg = W.get_config("C1", size=(16, 16, 16), weno_order=9)
    gg = PU.gpu_grid(binding, cfg)
    st = gg.fields_from_state(W.generate_state(cfg))
    G = PU.new_G(binding, gg, cfg)
    p = dict(cfg["params"]); p["adv_x"] = 7
    with pytest.raises(binding.OcnError) as e:
        binding.ocn_compute_tendencies(gg, p, st, None, G)
    assert e.value.code == binding.OCN_ERR_UNSUPPORTED
    p = dict(cfg["params"]); p["adv_y"] = 5
    with pytest.raises(binding.OcnError) as e:
        binding.ocn_compute_tendencies(gg, p, st, None, G)
    assert e.value.code == binding.OCN_ERR_UNSUPPORTED
    cfg3 = W.get_config("C1", size=(16, 16, 16))                       # halo 3
    g3 = PU.gpu_grid(binding, cfg3)
    st3 = g3.fields_from_state(W.generate_state(cfg3))
    G3 = PU.new_G(binding, g3, cfg3)
    p = dict(cfg3["params"]); p["adv_x"] = p["adv_y"] = p["adv_z"] = 7
    with pytest.raises(binding.OcnError) as e:
        binding.ocn_compute_tendencies(g3, p, st3, None, G3)
    assert e.value.code == binding.OCN_ERR_INVALID
    gg.set_kernel(2)
    with pytest.raises(binding.OcnError) as e:
        binding.ocn_compute_tendencies(gg, cfg["params"], st, None, G)
    assert e.value.code == binding.OCN_ERR_UNSUPPORTED


@pytest.mark.parametrize("order,dtype,eps_min", [(5, "f64", 1e-50), (7, "f64", 1e-38), (9, "f64", 1e-32), (9, "f32", 1e-30), (5, "f32", 1e-30)])
def test_smallest_weno_eps_on_constant_fields(binding, W, order, dtype, eps_min):
    """The WENO-Z weights are evaluated as products of the regularised indicators (fp64) / with flushed-denormal reciprocals (fp32):
    on a constant stencil an eps below the documented bound would give 0/0.  Below the bound the call is refused; AT the bound
    constant fields (every indicator exactly 0, the worst case) give finite, vanishing (fp64: exactly) advective tendencies."""
    cfg = dict(W.get_config("C1", size=(24, 20, 16), weno_order=order), dtype=dtype)
    gg = PU.gpu_grid(binding, cfg)
    state = W.generate_state(cfg)
    npdt = np.float64 if dtype == "f64" else np.float32
    const = {"u": 0.3, "v": -0.2, "w": 0.0}
    for k in ("u", "v", "w"):
        state[k] = np.full_like(state[k], const[k], dtype=npdt)
    state["c"] = [np.full_like(c, v, dtype=npdt) for c, v in zip(state["c"], (20.0, 35.0))]
    st = gg.fields_from_state(state)
    G = PU.new_G(binding, gg, cfg)
    p = dict(cfg["params"], weno_eps=eps_min * 0.5)
    with pytest.raises(binding.OcnError) as e:
        binding.ocn_compute_tendencies(gg, p, st, None, G)
    assert e.value.code == binding.OCN_ERR_INVALID and "weno_eps" in str(e.value)
    p = dict(cfg["params"], weno_eps=eps_min, f0=0.0, g=0.0)
    binding.ocn_fill_halos(gg, p, st)
    binding.ocn_compute_tendencies(gg, p, st, None, G)
    out = gg.state_from_fields(G)
    Hh = cfg["grid"]["halo"]
    for nm, a in PU.named(out):
        inner = a[Hh:-Hh, Hh:-Hh, Hh:-Hh]
        assert np.isfinite(inner).all(), "%s: NaN / inf with weno_eps = %g" % (nm, eps_min)
        if nm != "w":      # w = 0 on the walls makes w's own z-stencils non-constant; u, v, T, S are constant everywhere they are read
            assert np.abs(inner).max() <= (0.0 if dtype == "f64" else 1e-7), (nm, np.abs(inner).max())    # fp32: rounding residue of the flux differences
