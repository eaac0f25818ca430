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


@pytest.mark.parametrize("name,size,order", [("C0", None, 5), ("C1", (67, 35, 9), 5), ("C3", (48, 40, 12), 5), ("C4", (40, 24, 20), 5),
                                             ("C1", (40, 24, 20), 9)])
def test_elementwise_halo_kernel_stays_bitwise(binding, ref, W, name, size, order):
    """The per-element halo kernel (the reference implementation of the row-wise default) stays under test through the grid's
    diagnostic flag OCN_DIAG_HALO_ELEMENTWISE: halo fill bitwise equal to the oracle's, as in every other test."""
    cfg = W.get_config(name, weno_order=order) if size is None else W.get_config(name, size=size, weno_order=order)
    cfg = dict(cfg, diag=binding.OCN_DIAG_HALO_ELEMENTWISE)
    errs, *_ = PU.run_substage_parity(binding, ref, cfg, W.generate_state(cfg), kernel=0, stage=1)
    PU.assert_errs(errs, cfg["dtype"], "%s elementwise halo" % name)


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


# ------------------------------------------------------------------------------ H5: G_w without the constant b
def _zc_uniform(Nz, dz):
    return -dz * (Nz - np.arange(1, Nz + 1) + 0.5)


@pytest.mark.parametrize("kernel", KERNELS)
@pytest.mark.parametrize("name,size", [("C1", (40, 24, 20)), ("C1", (67, 35, 9)), ("C4", (40, 24, 20)), ("C4", (133, 37, 11))])
@pytest.mark.parametrize("variant", ["g0", "refprofiles"])
def test_gw_parity_without_the_constant_buoyancy(binding, ref, W, kernel, name, size, variant):
    """with T_ref = S_ref = 0 the constant b ~ -0.235 dominates max|G_w|, so the 1e-12 check tests the
    advection of w only to ~2e-10.  Here the same states with (a) g = 0 and (b) T_ref, S_ref = the background profiles
    (b reduces to the O(1e-6) anomaly): max|G_w| is then the advective / diffusive part itself."""
    cfg = W.get_config(name, size=size)
    p = dict(cfg["params"])
    if variant == "g0":
        p["g"] = 0.0
    else:
        zc = _zc_uniform(size[2], cfg["grid"]["dz_uniform"])
        p["T_ref"] = 20.0 + 0.01 * zc
        p["S_ref"] = np.full(size[2], 35.0)
    cfg = dict(cfg, params=p)
    state = W.generate_state(cfg)
    prev = None
    for stage in (1, 2):
        errs, new_gpu, (Gf, G64), gg = PU.run_substage_parity(binding, ref, cfg, state, kernel=kernel, stage=stage, G_prev_pair=prev)
        PU.assert_errs(errs, cfg["dtype"], "%s %s stage %d kernel %d" % (name, variant, stage, kernel))
        # the point of the test: the scale of G_w is no longer the constant b
        gw = np.abs(PU.ref_grid(ref, cfg).interior(np.asarray(G64["w"]))).max()
        assert gw < 5e-3, gw
        prev = (Gf, G64)
        state = new_gpu


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


def _interior_equal(rg, a, b):
    return np.array_equal(rg.interior(np.asarray(a)), rg.interior(np.asarray(b)))


@pytest.mark.parametrize("name,size,kernel", [("C1", (40, 24, 20), 0), ("C1", (67, 35, 9), 0), ("C2", (64, 48, 32), 0), ("C3", (48, 40, 12), 0),
                                              ("C3", (71, 33, 50), 0), ("C4", (40, 24, 20), 0), ("C4", (133, 37, 11), 0),
                                              # the general per-cell kernel with the substage fused in: C0 (2-D, prescribed velocities) and
                                              # OCN_KERNEL_PERCELL on the 3-D workloads
                                              ("C0", None, 0), ("C1", (67, 35, 9), 1), ("C3", (48, 40, 12), 1), ("C4", (40, 24, 20), 1)])
def test_tendencies_rk3_is_bit_identical_to_the_two_calls(binding, ref, W, name, size, kernel):
    """ocn_tendencies_rk3 (tendencies + (A4) in one pass, ping-pong state) == ocn_compute_tendencies followed by
    ocn_rk3_substage, bit for bit, for G and for the state, at every stage."""
    import torch
    cfg = W.get_config(name) if size is None else W.get_config(name, size=size)
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
            assert _interior_equal(rg, x, y), "%s stage %d: G_%s differs" % (name, stage, nm)
        for (nm, x), (_, y) in zip(PU.named(sa), PU.named(sb)):
            if nm == "w" and p["hydrostatic"]:
                continue
            assert _interior_equal(rg, x, y), "%s stage %d: state %s differs" % (name, stage, nm)
        Ga, Gpa = Gpa, Ga
        Gb, Gpb = Gpb, Gb
        b, b2 = b2, b


@pytest.mark.parametrize("name,size", [("C1", (40, 24, 20)), ("C3", (48, 40, 12)), ("C3", (71, 33, 50)), ("C4", (40, 24, 20)), ("C0", None)])
def test_step_fused_matches_step(binding, ref, W, name, size):
    """ocn_step_fused == ocn_step bit for bit.  On the hydrostatic workload this also checks the w that the TMA-ring kernel diagnoses
    from continuity by itself (ocn_step_fused does not launch ocn_compute_w) against the column-scan kernel ocn_step uses."""
    import torch
    cfg = W.get_config(name) if size is None else W.get_config(name, size=size)
    p = cfg["params"]
    rg = PU.ref_grid(ref, cfg)
    gg = PU.gpu_grid(binding, cfg)
    state = W.generate_state(cfg)
    a, b = gg.fields_from_state(state), gg.fields_from_state(state)
    b2 = gg.fields(n_tracers=p["n_tracers"], w=state.get("w") is not None)
    if not p["momentum_prognostic"]:                      # prescribed velocities are shared by the ping-pong pair
        b2.u, b2.v, b2.w = b.u, b.v, b.w
    G, Gp = PU.new_G(binding, gg, cfg), PU.new_G(binding, gg, cfg)
    phy = gg.new_field() if p["hydrostatic"] else None
    binding.ocn_step(gg, p, 3, cfg["dt"], a, G, Gp, phy)
    binding.ocn_step_fused(gg, p, 3, cfg["dt"], b, b2, G, Gp, phy)
    torch.cuda.synchronize()
    for (nm, x), (_, y) in zip(PU.named(gg.state_from_fields(a)), PU.named(gg.state_from_fields(b2))):
        if nm == "w" and p["hydrostatic"]:
            continue
        assert _interior_equal(rg, x, y), "%s: state %s differs between ocn_step and ocn_step_fused" % (name, nm)


def test_fused_entry_points_refuse_what_the_fused_kernel_does_not_cover(binding, W):
    # every model has a kernel with the substage fused in; what is refused is the TMA-ring kernel forced (OCN_KERNEL_FUSED) on a model it does not cover
    cfg = W.get_config("C0")
    p = cfg["params"]
    gg = PU.gpu_grid(binding, cfg, 2)
    st = gg.fields_from_state(W.generate_state(cfg))
    alt = gg.fields(n_tracers=1, w=False)
    alt.u, alt.v = st.u, st.v
    G = PU.new_G(binding, gg, cfg)
    with pytest.raises(binding.OcnError) as e:
        binding.ocn_tendencies_rk3(gg, p, 1, cfg["dt"], st, None, G, None, alt)
    assert e.value.code == binding.OCN_ERR_UNSUPPORTED
    cfg = W.get_config("C1", size=(40, 24, 20))
    p = cfg["params"]
    gg = PU.gpu_grid(binding, cfg)
    st = gg.fields_from_state(W.generate_state(cfg))
    G = PU.new_G(binding, gg, cfg)
    with pytest.raises(binding.OcnError) as e:      # in place is not allowed
        binding.ocn_tendencies_rk3(gg, p, 1, cfg["dt"], st, None, G, None, st)
    assert e.value.code == binding.OCN_ERR_INVALID
    with pytest.raises(binding.OcnError) as e:      # stage 2 needs G_prev
        binding.ocn_tendencies_rk3(gg, p, 2, cfg["dt"], st, None, G, None, gg.fields(n_tracers=2))
    assert e.value.code == binding.OCN_ERR_INVALID


@pytest.mark.parametrize("fused", [False, True])
def test_step_host_matches_step(binding, ref, W, fused):
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
    alt = gg.fields(n_tracers=p["n_tracers"]) if fused else None
    binding.ocn_step_host(gg, p, 3, cfg["dt"], host, dev2, alt, G, Gp, None)
    torch.cuda.synchronize()
    L = gg.layout
    for nm, t in (("u", host.u), ("v", host.v), ("w", host.w), ("c0", host.c[0]), ("c1", host.c[1])):
        a = t.view(L.nz_pad, L.ny_pad, L.stride_y)[:, :, gg._xo:gg._xo + L.nx_pad].numpy()
        b = want[nm] if nm in want else want["c"][int(nm[1:])]
        assert np.array_equal(PU.ref_grid(ref, cfg).interior(a), PU.ref_grid(ref, cfg).interior(b)), nm
