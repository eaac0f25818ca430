"""GPU parity of SURVEY 8(f) N3, vertically-implicit diffusion (A2) PAPER.md:785-803 / (A8) PAPER.md:829-835, through the C ABI.

(1) With ocn_params.implicit_vertical_diffusion = 1 the tendency kernels (per-cell, fused, high-order) must leave the
    vertical diffusion out of G: compared with the oracle's tendencies computed with the same flag, north_star tolerances.
(2) ocn_implicit_vertical_diffusion is compared element by element with the oracle's long-double Thomas solve of THE SAME
    input arrays (teacher-forced), relative to max|field|: 1e-12 (fp64) / 2e-5 (fp32).
(3) The whole substage {halos, tendencies(flag), RK3 substage, implicit solve} chained on the GPU vs the oracle's chain."""
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


def _implicit_cfg(W, name, size, nu=None, kappa=None, weno_order=5):
    cfg = W.get_config(name, size=size, weno_order=weno_order)
    p = dict(cfg["params"], implicit_vertical_diffusion=1)
    if nu is not None:
        p["nu"] = nu
    if kappa is not None:
        p["kappa"] = list(kappa) + [0.0] * (8 - len(kappa))
    return dict(cfg, params=p)


CASES = [("C1", (40, 24, 20), 0, 5), ("C1", (40, 24, 20), 1, 5), ("C1", (67, 35, 9), 2, 5), ("C3", (48, 40, 12), 0, 5),
         ("C3", (71, 33, 50), 1, 5), ("C4", (40, 24, 20), 0, 5), ("C4", (133, 37, 11), 1, 5), ("C1", (40, 24, 20), 0, 7),
         ("C1", (40, 24, 20), 1, 9)]


@pytest.mark.parametrize("name,size,kernel,order", CASES)
def test_tendencies_leave_out_vertical_diffusion(binding, ref, name, size, kernel, order):
    from paper_2502_14148_b200 import workloads as W
    # a diffusivity large enough for the dropped term to matter in G at these tolerances
    ntr = W.get_config(name, size=size)["params"]["n_tracers"]
    cfg = _implicit_cfg(W, name, size, nu=3e-3, kappa=[2e-3, 5e-3, 1e-3][:ntr], weno_order=order)
    if kernel == 2 and name == "C3":
        pytest.skip("covered by kernel 0")
    errs, *_ = PU.run_substage_parity(binding, ref, cfg, W.generate_state(cfg), kernel=kernel, stage=1)
    PU.assert_errs(errs, cfg["dtype"], "implicit-flag tendencies %s %s k%d o%d" % (name, size, kernel, order))
    # and the flag really changes G (guards against both sides ignoring it)
    cfg_e = dict(cfg, params=dict(cfg["params"], implicit_vertical_diffusion=0))
    rg = PU.ref_grid(ref, cfg)
    st = PU.to64(W.generate_state(cfg))
    ref.fill_halos(rg, cfg["params"], st)
    if cfg["params"]["hydrostatic"]:
        ref.compute_w(rg, st)
    ph = ref.compute_phy(rg, cfg["params"], st) if cfg["params"]["hydrostatic"] else None
    Gi = ref.compute_tendencies(rg, cfg["params"], st, ph)
    Ge = ref.compute_tendencies(rg, cfg_e["params"], st, ph)
    assert np.abs(rg.interior(Gi["c"][0]) - rg.interior(Ge["c"][0])).max() > 1e-6 * np.abs(rg.interior(Ge["c"][0])).max()


def _solve_parity(B, ref, cfg, state, dt, tol):
    rg, gg = PU.ref_grid(ref, cfg), PU.gpu_grid(B, cfg)
    p = cfg["params"]
    st = gg.fields_from_state(state)
    B.ocn_implicit_vertical_diffusion(gg, p, dt, st)
    got = gg.state_from_fields(st)
    want = PU.copy_state(PU.to64(state))          # to64 does not copy float64 arrays
    ref.implicit_vertical_diffusion(rg, p, dt, want)
    errs = {}
    for (nm, a), (_, b) in zip(PU.named(got), PU.named(want)):
        errs[nm], _ = PU.rel_err(rg, a, b)
        m = np.ones(rg.shape, bool)
        rg.interior(m)[...] = False
        src = state[nm] if nm in ("u", "v", "w") else state["c"][int(nm[1:])]
        assert np.array_equal(a[m], src[m]), "halo of %s was touched" % nm
    bad = {k: v for k, v in errs.items() if not v <= tol}
    assert not bad, "beyond %.0e: %s (all %s)" % (tol, bad, errs)
    return got, want


@pytest.mark.parametrize("name,size,dt", [("C1", (16, 8, 300), 50.0),      # taller than the shared-memory tile: the global-sweep kernel
                                          ("C1", (8, 8, 2100), 50.0),      # taller than the block-parallel pivots kernel's shared memory: serial pivots
                                          ("C1", (40, 24, 20), 50.0), ("C1", (67, 35, 9), 4.0), ("C1", (128, 128, 64), 300.0),
                                          ("C3", (48, 40, 12), 2.0e4), ("C3", (71, 33, 50), 3.0e5), ("C4", (40, 24, 20), 50.0),
                                          ("C4", (133, 37, 11), 7.0)])
def test_implicit_solve_teacher_forced(binding, ref, name, size, dt):
    from paper_2502_14148_b200 import workloads as W
    ntr = W.get_config(name, size=size)["params"]["n_tracers"]
    cfg = _implicit_cfg(W, name, size, nu=0.3, kappa=[0.7, 0.2, 0.05][:ntr])
    state = W.generate_state(cfg)
    rg = PU.ref_grid(ref, cfg)
    if cfg["params"]["hydrostatic"]:             # w is diagnosed: give it values so that "not touched" is a real check
        state["w"] = np.random.default_rng(1).standard_normal(rg.shape).astype(state["u"].dtype)
    got, want = _solve_parity(binding, ref, cfg, state, dt, PU.TOL[cfg["dtype"]])
    if cfg["params"]["hydrostatic"]:
        assert np.array_equal(got["w"], state["w"])
    # the solve is far from the identity at these dt*kz/dz^2
    assert np.abs(rg.interior(got["c"][0]).astype(np.float64) - rg.interior(state["c"][0])).max() > 1e-4 * np.abs(rg.interior(state["c"][0])).max()


def test_zero_diffusivity_fields_are_skipped_bitwise(binding, ref):
    from paper_2502_14148_b200 import workloads as W
    cfg = _implicit_cfg(W, "C1", (40, 24, 20), nu=0.0, kappa=[0.0, 0.4])
    state = W.generate_state(cfg)
    got, _ = _solve_parity(binding, ref, cfg, state, 10.0, 1e-12)
    for nm in ("u", "v", "w"):
        assert np.array_equal(got[nm], state[nm])
    assert np.array_equal(got["c"][0], state["c"][0])
    assert not np.array_equal(got["c"][1], state["c"][1])


@pytest.mark.parametrize("name,size", [("C1", (40, 24, 20)), ("C4", (40, 24, 20))])
def test_chained_substage_with_implicit_diffusion(binding, ref, name, size):
    """{fill halos, tendencies (flag), RK3 substage, implicit solve} on the GPU vs the oracle's own chain from the same
    initial state: state fields only (protocol P2)."""
    from paper_2502_14148_b200 import workloads as W
    B = binding
    ntr = W.get_config(name, size=size)["params"]["n_tracers"]
    cfg = _implicit_cfg(W, name, size, nu=0.05, kappa=[0.08, 0.02, 0.01][:ntr])
    p, dt = cfg["params"], cfg["dt"]
    rg, gg = PU.ref_grid(ref, cfg), PU.gpu_grid(B, cfg)
    state = W.generate_state(cfg)
    st = gg.fields_from_state(state)
    G = PU.new_G(B, gg, cfg)
    B.ocn_fill_halos(gg, p, st)
    B.ocn_compute_tendencies(gg, p, st, None, G)
    B.ocn_rk3_substage(gg, p, 1, dt, st, G, None)
    B.ocn_implicit_vertical_diffusion(gg, p, dt * 8.0 / 15.0, st)
    got = gg.state_from_fields(st)
    rs = PU.to64(state)
    ref.fill_halos(rg, p, rs)
    Gr = ref.compute_tendencies(rg, p, rs)
    ref.rk3_substage(rg, p, 1, dt, rs, Gr, None)
    ref.implicit_vertical_diffusion(rg, p, dt * 8.0 / 15.0, rs)
    tol = 1e-12 if cfg["dtype"] == "f64" else 2e-5
    for (nm, a), (_, b) in zip(PU.named(got), PU.named(rs)):
        e, _ = PU.rel_err(rg, a, b)
        assert e <= tol, (nm, e)


def test_invalid_arguments(binding):
    from paper_2502_14148_b200 import workloads as W
    B = binding
    cfg = W.get_config("C0")
    gg = PU.gpu_grid(B, cfg)
    st = gg.fields_from_state(W.generate_state(cfg))
    with pytest.raises(B.OcnError) as e:
        B.ocn_implicit_vertical_diffusion(gg, cfg["params"], 1.0, st)       # z is Flat
    assert e.value.code == B.OCN_ERR_INVALID
    cfg = W.get_config("C1", size=(40, 24, 20))
    gg = PU.gpu_grid(B, cfg)
    st = gg.fields(n_tracers=2)
    with pytest.raises(B.OcnError) as e:
        B.ocn_implicit_vertical_diffusion(gg, cfg["params"], -1.0, st)
    assert e.value.code == B.OCN_ERR_INVALID
    with pytest.raises(B.OcnError) as e:
        B.ocn_implicit_vertical_diffusion(gg, dict(cfg["params"], nu=-1.0), 1.0, st)
    assert e.value.code == B.OCN_ERR_INVALID


@pytest.mark.parametrize("name", ["C2", "C4"])
def test_fullsize_implicit_solve_inverts_the_operator(binding, name):
    """BASELINE sizes (C2 512x512x256 fp64, C4 1024x1024x128 fp32) in the launch configuration bench.py times: a property
    that holds at any size — applying (1 - dt kz d_z d_z) (torch slicing, no-flux walls / w = 0 on the walls) to the result
    gives back the input — on the tracer T and on w."""
    import torch
    from paper_2502_14148_b200 import workloads as W
    B = binding
    cfg = W.get_config(name)
    g = cfg["grid"]
    p = dict(cfg["params"], implicit_vertical_diffusion=1, nu=0.3, kappa=[0.7, 0.2, 0.05] + [0.0] * 5)
    gg = PU.gpu_grid(B, cfg)
    tdt = gg.tdtype
    gen = torch.Generator(device="cuda").manual_seed(11)
    st = gg.fields(n_tracers=1)
    shape = (g["Nz"], g["Ny"], g["Nx"])
    for t in (st.w, st.c[0]):
        gg.interior(t).copy_(torch.randn(shape, device="cuda", dtype=tdt, generator=gen))
    gg.interior(st.w)[0] = 0
    old_c = gg.interior(st.c[0]).double().clone()
    old_w = gg.interior(st.w).double().clone()
    p1 = dict(p, n_tracers=1, idx_T=0, idx_S=-1)
    dt, dz = 3.0, g["dz_uniform"]
    B.ocn_implicit_vertical_diffusion(gg, p1, dt, st)
    c = gg.interior(st.c[0]).double()
    flux = torch.zeros((shape[0] + 1,) + shape[1:], device="cuda", dtype=torch.float64)
    flux[1:-1] = (c[1:] - c[:-1]) / dz
    back = c - dt * 0.7 * (flux[1:] - flux[:-1]) / dz
    tol = 1e-12 if cfg["dtype"] == "f64" else 2e-5
    assert (back - old_c).abs().max().item() <= tol * 10 * old_c.abs().max().item()
    del flux, back
    w = gg.interior(st.w).double()                      # faces 1..Nz, face 1 and the implicit face Nz+1 are walls (0)
    wf = torch.cat([w, torch.zeros_like(w[:1])], 0)
    d = (wf[1:] - wf[:-1]) / dz                         # at centres 1..Nz
    lap = torch.zeros_like(w)
    lap[1:] = (d[1:] - d[:-1]) / dz
    back = w - dt * 0.3 * lap
    assert (back - old_w).abs().max().item() <= tol * 10 * old_w.abs().max().item()
    assert gg.interior(st.w)[0].abs().max().item() == 0.0
