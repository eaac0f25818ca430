"""ocn_step_model (include/ocn.h): one time step of a complete model = the hot path + the SURVEY 8(f) rows the options select.
(1) bit-identical to the same sequence of individual C-ABI calls issued from Python; (2) protocol P2 (state after a full step)
against the oracle's own chain {fill halos, tendencies, RK3 substage, [implicit solve], [barotropic substeps + correction],
[pressure correction]} from the same initial state, at the north_star tolerances."""
import numpy as np
import pytest

from tests import parity_util as PU

pytestmark = pytest.mark.gpu
GAM = (8.0 / 15.0, 5.0 / 12.0, 3.0 / 4.0)
ZET = (0.0, 17.0 / 60.0, 5.0 / 12.0)


@pytest.fixture(scope="module")
def binding():
    import torch
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    from paper_2502_14148_b200 import binding as Bd
    Bd.lib()
    return Bd


def _alt(B, gg, st, hydro):
    return B.Fields(gg.new_field(), gg.new_field(), st.w if hydro else gg.new_field(), [gg.new_field() for _ in st.c])


def _python_chain(B, gg, p, dt, st, alt, G, Gp, phy, poisson=None, p_nh=None, bt=None, bt_N=0, wts=None):
    cur, nxt, Gm, Gq = st, alt, G, Gp
    hydro = bool(p["hydrostatic"])
    for m in (1, 2, 3):
        share = GAM[m - 1] - ZET[m - 1]
        B.ocn_fill_halos(gg, p, cur)
        if hydro:
            B.ocn_compute_w(gg, cur)
            B.ocn_compute_phy(gg, p, cur, phy)
        B.ocn_tendencies_rk3(gg, p, m, dt, cur, phy, Gm, None if m == 1 else Gq, nxt)
        if p.get("implicit_vertical_diffusion"):
            B.ocn_implicit_vertical_diffusion(gg, p, dt * share, nxt)
        if bt is not None:
            B.ocn_barotropic_forcing(gg, GAM[m - 1] / share, ZET[m - 1] / share, Gm, None if m == 1 else Gq, bt)
            B.ocn_barotropic_substeps(gg, p["g"], dt * share, bt_N, wts, bt)
            B.ocn_barotropic_correct(gg, nxt, bt)
        if poisson is not None:
            B.ocn_pressure_correction(poisson, dt * share, nxt, p_nh)
        cur, nxt, Gm, Gq = nxt, cur, Gq, Gm
    return cur


@pytest.mark.parametrize("implicit", [0, 1])
def test_nonhydrostatic_step_with_projection(binding, ref, implicit):
    from paper_2502_14148_b200 import workloads as W
    B = binding
    cfg = W.get_config("C1", size=(40, 24, 20))
    p = dict(cfg["params"], implicit_vertical_diffusion=implicit, nu=0.02, kappa=[0.03, 0.01] + [0.0] * 6)
    dt = cfg["dt"]
    rg, gg = PU.ref_grid(ref, cfg), PU.gpu_grid(B, cfg)
    state = W.generate_state(cfg)
    res = []
    for use_model in (True, False):
        st = gg.fields_from_state(state)
        alt = _alt(B, gg, st, False)
        G, Gp = PU.new_G(B, gg, cfg), PU.new_G(B, gg, cfg)
        ps, p_nh = B.ocn_poisson_create(gg), gg.new_field()
        if use_model:
            B.ocn_step_model(gg, p, 3, dt, st, alt, G, Gp, poisson=ps, p_nh=p_nh)
            out = alt
        else:
            out = _python_chain(B, gg, p, dt, st, alt, G, Gp, None, poisson=ps, p_nh=p_nh)
        res.append(gg.state_from_fields(out))
    for (nm, a), (_, b) in zip(PU.named(res[0]), PU.named(res[1])):
        assert np.array_equal(rg.interior(a), rg.interior(b)), nm
    # oracle chain (P2)
    rs = PU.to64(PU.copy_state(state))
    Gr_prev = None
    for m in (1, 2, 3):
        share = GAM[m - 1] - ZET[m - 1]
        ref.fill_halos(rg, p, rs)
        Gr = ref.compute_tendencies(rg, p, rs)
        ref.rk3_substage(rg, p, m, dt, rs, Gr, Gr_prev)
        if implicit:
            ref.implicit_vertical_diffusion(rg, p, dt * share, rs)
        ref.pressure_correction(rg, dt * share, rs)
        Gr_prev = Gr
    for (nm, a), (_, b) in zip(PU.named(res[0]), PU.named(rs)):
        e, _ = PU.rel_err(rg, a, b)
        assert e <= 1e-12, (nm, e)
    # the step ends discretely solenoidal
    d = ref.divergence(rg, PU.to64(res[0]))
    assert np.abs(rg.interior(d)).max() <= 1e-15


def test_hydrostatic_step_with_free_surface(binding, ref):
    from paper_2502_14148_b200 import workloads as W
    B = binding
    cfg = W.get_config("C3", size=(71, 33, 50))
    p = dict(cfg["params"], implicit_vertical_diffusion=1)
    dt = cfg["dt"]
    rg, gg = PU.ref_grid(ref, cfg), PU.gpu_grid(B, cfg)
    state = W.generate_state(cfg)
    N = 12
    wts = W.barotropic_weights(N)
    res = []
    for use_model in (True, False):
        st = gg.fields_from_state(state)
        alt = _alt(B, gg, st, True)
        G, Gp = PU.new_G(B, gg, cfg), PU.new_G(B, gg, cfg)
        phy = gg.new_field()
        bt = B.Barotropic(gg)
        B.ocn_barotropic_init(gg, st, bt)
        if use_model:
            B.ocn_step_model(gg, p, 3, dt, st, alt, G, Gp, p_hy=phy, bt=bt, bt_N=N, bt_weights=wts)
            out = alt
        else:
            out = _python_chain(B, gg, p, dt, st, alt, G, Gp, phy, bt=bt, bt_N=N, wts=wts)
        res.append((gg.state_from_fields(out), {k: bt.download(getattr(bt, k)) for k in ("eta", "U", "V")}))
    for (nm, a), (_, b) in zip(PU.named(res[0][0]), PU.named(res[1][0])):
        if nm != "w":
            assert np.array_equal(rg.interior(a), rg.interior(b)), nm
    for k in ("eta", "U", "V"):
        assert np.array_equal(res[0][1][k], res[1][1][k]), k
    # oracle chain (P2): state fields and barotropic variables
    rs = PU.to64(PU.copy_state(state))
    ref.fill_halos(rg, p, rs)
    rbt = ref.barotropic_init(rg, rs)
    Gr_prev = None
    for m in (1, 2, 3):
        share = GAM[m - 1] - ZET[m - 1]
        ref.fill_halos(rg, p, rs)
        ref.compute_w(rg, rs)
        ph = ref.compute_phy(rg, p, rs)
        Gr = ref.compute_tendencies(rg, p, rs, ph)
        ref.rk3_substage(rg, p, m, dt, rs, Gr, Gr_prev)
        ref.implicit_vertical_diffusion(rg, p, dt * share, rs)
        FU, FV = ref.barotropic_forcing(rg, GAM[m - 1] / share, ZET[m - 1] / share, Gr, Gr_prev)
        ref.barotropic_substeps(rg, p["g"], dt * share, N, wts, rbt, FU, FV)
        ref.barotropic_correct(rg, rs, rbt)
        Gr_prev = Gr
    for (nm, a), (_, b) in zip(PU.named(res[0][0]), PU.named(rs)):
        if nm == "w":
            continue
        e, _ = PU.rel_err(rg, a, b)
        assert e <= 1e-11, (nm, e)
    for k in ("eta", "U", "V"):
        den = np.abs(rbt[k]).max()
        assert np.abs(res[0][1][k] - rbt[k]).max() <= 1e-10 * den, k


def test_option_errors(binding):
    from paper_2502_14148_b200 import workloads as W
    B = binding
    cfg = W.get_config("C3", size=(48, 40, 12))
    gg = PU.gpu_grid(B, cfg)
    st = gg.fields_from_state(W.generate_state(cfg))
    alt = _alt(B, gg, st, True)
    G, Gp = PU.new_G(B, gg, cfg), PU.new_G(B, gg, cfg)
    c1 = W.get_config("C1", size=(48, 40, 12))
    g1 = PU.gpu_grid(B, c1)
    ps = B.ocn_poisson_create(g1)
    with pytest.raises(B.OcnError) as e:          # pressure correction on a hydrostatic model
        B.ocn_step_model(gg, cfg["params"], 3, 1.0, st, alt, G, Gp, p_hy=gg.new_field(), poisson=ps, p_nh=gg.new_field())
    assert e.value.code == B.OCN_ERR_INVALID
    with pytest.raises(B.OcnError) as e:
        B.ocn_step_model(gg, cfg["params"], 4, 1.0, st, alt, G, Gp, p_hy=gg.new_field())
    assert e.value.code == B.OCN_ERR_INVALID


def test_solver_must_belong_to_the_grid_and_buffers_must_be_aligned(binding):
    """a Poisson solver built for another grid (or whose grid is gone) is refused before anything is enqueued;
    a field buffer that is not aligned to ocn_layout.alignment_bytes gives OCN_ERR_INVALID instead of a device fault."""
    import torch
    from paper_2502_14148_b200 import workloads as W
    B = binding
    cfg = W.get_config("C1", size=(40, 24, 20))
    p = cfg["params"]
    gg = PU.gpu_grid(B, cfg)
    other = PU.gpu_grid(B, W.get_config("C1", size=(48, 40, 12)))
    st = gg.fields_from_state(W.generate_state(cfg))
    alt = _alt(B, gg, st, False)
    G, Gp = PU.new_G(B, gg, cfg), PU.new_G(B, gg, cfg)
    before = gg.state_from_fields(st)
    ps_other = B.ocn_poisson_create(other)
    n0 = B.ocn_launch_count()
    with pytest.raises(B.OcnError) as e:
        B.ocn_step_model(gg, p, 3, 0.1, st, alt, G, Gp, poisson=ps_other, p_nh=gg.new_field())
    assert e.value.code == B.OCN_ERR_INVALID and "another grid" in str(e.value)
    with pytest.raises(B.OcnError) as e:          # dt <= 0 with a pressure correction: caught before substage 1 runs
        B.ocn_step_model(gg, p, 3, 0.0, st, alt, G, Gp, poisson=B.ocn_poisson_create(gg), p_nh=gg.new_field())
    assert e.value.code == B.OCN_ERR_INVALID
    assert B.ocn_launch_count() == n0, "a kernel was enqueued before the argument error was reported"
    torch.cuda.synchronize()
    for (nm, a), (_, b) in zip(PU.named(before), PU.named(gg.state_from_fields(st))):
        assert np.array_equal(a, b), nm
    # the solver of a destroyed grid
    tmp = PU.gpu_grid(B, cfg)
    ps_tmp = B.ocn_poisson_create(tmp)
    B.lib().ocn_grid_destroy(tmp._h)
    tmp._h = None
    with pytest.raises(B.OcnError) as e:
        B.ocn_pressure_correction(ps_tmp, 0.1, st, gg.new_field())
    assert e.value.code == B.OCN_ERR_INVALID and "destroyed" in str(e.value)
    # misaligned field buffer: a view 8 bytes into an allocation
    raw = torch.zeros(gg.layout.n_alloc + 16, dtype=torch.float64, device="cuda")
    bad = B.Fields(raw[1:1 + gg.layout.n_alloc], st.v, st.w, list(st.c))
    with pytest.raises(B.OcnError) as e:
        B.ocn_fill_halos(gg, p, bad)
    assert e.value.code == B.OCN_ERR_INVALID and "aligned" in str(e.value)
