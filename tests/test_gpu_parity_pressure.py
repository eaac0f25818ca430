"""GPU parity of SURVEY 8(f) N2, the pressure correction (A8)-(A12) PAPER.md:829-851, through the C ABI.

P1 teacher-forced, call by call: ocn_pressure_rhs vs the oracle's divergence of the SAME predictor; ocn_poisson_solve vs the
oracle's long-double eigenfunction-expansion solve of the GPU's OWN right-hand side; ocn_pressure_correct vs (A11) applied to
the GPU's own p.  Then the composed call against the oracle's end-to-end long-double correction, and the defining property
div(u^{m+1}) = 0 (checked with numpy rolls, at any size).

Tolerances.  u, v, w: the north_star's 1e-12 (fp64) / 2e-5 (fp32) relative to max|field|.  p and rhs: the same numbers
relative to max|p| / max|rhs| when the predictor has O(1) divergence (random velocity).  For a hot-path predictor (a
solenoidal state plus one substage increment) div(u~) is a small difference of O(|u|/dx) terms, so rhs and p are compared in the
backward-error form |err| <= tol * max|u| / (dx dt) (rhs) and tol * max|u| dx / dt (p): DESIGN.md 7."""
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


def _cfg(W, name, size):
    return W.get_config(name, size=size)


def _custom_cfg(W, Nx, Ny, Nz, dtype="f64", stretched=False, flat_z=False, dx=1.0, dy=1.0):
    cfg = W.get_config("C1", size=(Nx, Ny, max(Nz, 3)))
    g = dict(cfg["grid"])
    if flat_z:
        g.update(Nz=1, topology=(0, 0, 2), dz_c=None, dz_uniform=1.0)
    elif stretched:
        r = np.random.default_rng(5)
        g.update(Nz=Nz, dz_c=(0.5 + 1.5 * r.random(Nz)), dz_uniform=1.0)
    g.update(dx=dx, dy=dy)
    cfg = dict(cfg, grid=g, dtype=dtype)
    return cfg


def _random_velocity(rg, dtype, seed, flat_z=False):
    r = np.random.default_rng(seed)
    npdt = np.float64 if dtype == "f64" else np.float32
    st = {"u": None, "v": None, "w": None, "c": []}
    for nm in ("u", "v", "w"):
        if nm == "w" and flat_z:
            continue
        a = np.zeros(rg.shape, dtype=npdt)
        rg.interior(a)[...] = r.standard_normal((rg.Nz, rg.Ny, rg.Nx)).astype(npdt)
        if nm == "w":
            rg.interior(a)[0] = 0
        st[nm] = a
    return st


def _np_div(rg, st, dz):
    u, v = rg.interior(st["u"]).astype(np.float64), rg.interior(st["v"]).astype(np.float64)
    d = (np.roll(u, -1, axis=2) - u) / rg.dx + (np.roll(v, -1, axis=1) - v) / rg.dy
    if st.get("w") is not None:
        w = rg.interior(st["w"]).astype(np.float64)
        wf = np.concatenate([w, np.zeros((1,) + w.shape[1:])], axis=0)
        wf[0] = 0
        d += np.diff(wf, axis=0) / dz[:, None, None]
    return d


def _call_by_call(B, ref, cfg, state, dt, tol, hot=False):
    rg, gg = PU.ref_grid(ref, cfg), PU.gpu_grid(B, cfg)
    flat = cfg["grid"]["topology"][2] == 2
    ps = B.ocn_poisson_create(gg)
    st = gg.fields_from_state(state)
    s64 = PU.to64(state)
    umax = max(np.abs(a).max() for _, a in PU.named(s64))
    dmin = min(rg.dx, rg.dy)
    errs = {}
    # rhs
    rhs = gg.new_field()
    B.ocn_pressure_rhs(gg, dt, st, rhs)
    rhs_gpu = gg.download(rhs)
    rhs_ref = ref.divergence(rg, s64, 1.0 / dt)
    den = umax / (dmin * dt) if hot else np.abs(rhs_ref).max()
    errs["rhs"] = np.abs(rg.interior(rhs_gpu.astype(np.float64)) - rg.interior(rhs_ref)).max() / den
    # solve, teacher-forced on the GPU's rhs
    p = gg.new_field()
    B.ocn_poisson_solve(ps, rhs, p)
    p_gpu = gg.download(p)
    p_ref = ref.poisson_solve(rg, rhs_gpu.astype(np.float64))
    den = umax * dmin / dt if hot else np.abs(p_ref).max()
    errs["p"] = np.abs(rg.interior(p_gpu.astype(np.float64)) - rg.interior(p_ref)).max() / den
    # in place (rhs aliases p) gives the same bits
    B.ocn_poisson_solve(ps, rhs, rhs)
    assert np.array_equal(gg.download(rhs), p_gpu)
    # correct, teacher-forced on the GPU's p
    B.ocn_pressure_correct(gg, dt, st, p)
    new_gpu = gg.state_from_fields(st)
    new_ref = PU.copy_state(s64)
    ref.pressure_correct(rg, dt, new_ref, p_gpu.astype(np.float64))
    for nm in ("u", "v", "w"):
        if new_ref[nm] is not None:
            errs["q_" + nm] = np.abs(rg.interior(new_gpu[nm].astype(np.float64)) - rg.interior(new_ref[nm])).max() / umax
    # halos untouched by the correction
    for nm in ("u", "v", "w"):
        if state[nm] is not None:
            m = np.ones(rg.shape, bool)
            rg.interior(m)[...] = False
            assert np.array_equal(new_gpu[nm][m], state[nm][m])
    # the defining property, by numpy
    dz = rg.metric("dzc") if not flat else np.ones(1)
    d1 = np.abs(_np_div(rg, new_gpu, dz)).max()
    eps = 2.3e-16 if cfg["dtype"] == "f64" else 1.2e-7
    assert d1 <= 100 * eps * umax / dmin, ("div after correction", d1, umax / dmin)
    bad = {k: v for k, v in errs.items() if not v <= tol}
    assert not bad, "beyond %.0e: %s (all %s)" % (tol, bad, errs)
    return errs


SIZES64 = [(40, 24, 20), (67, 35, 9), (128, 128, 64)]


@pytest.mark.parametrize("size", SIZES64)
def test_random_velocity_call_by_call_f64(binding, ref, size):
    from paper_2502_14148_b200 import workloads as W
    cfg = _cfg(W, "C1", size)
    rg = PU.ref_grid(ref, cfg)
    _call_by_call(binding, ref, cfg, _random_velocity(rg, "f64", 3), 0.37, 1e-12)


@pytest.mark.parametrize("size", [(40, 24, 20), (133, 37, 11)])
def test_random_velocity_call_by_call_f32(binding, ref, size):
    from paper_2502_14148_b200 import workloads as W
    cfg = _cfg(W, "C4", size)
    rg = PU.ref_grid(ref, cfg)
    _call_by_call(binding, ref, cfg, _random_velocity(rg, "f32", 4), 0.37, 2e-5)


def test_stretched_z_and_anisotropic_spacing(binding, ref):
    from paper_2502_14148_b200 import workloads as W
    cfg = _custom_cfg(W, 36, 30, 17, stretched=True, dx=0.5, dy=2.0)
    rg = PU.ref_grid(ref, cfg)
    _call_by_call(binding, ref, cfg, _random_velocity(rg, "f64", 6), 1.3, 1e-12)


def test_flat_z_two_dimensional(binding, ref):
    from paper_2502_14148_b200 import workloads as W
    cfg = _custom_cfg(W, 64, 48, 1, flat_z=True)
    rg = PU.ref_grid(ref, cfg)
    _call_by_call(binding, ref, cfg, _random_velocity(rg, "f64", 7, flat_z=True), 0.1, 1e-12)


@pytest.mark.parametrize("name,size,tol", [("C1", (40, 24, 20), 1e-12), ("C1", (128, 128, 64), 1e-12), ("C4", (40, 24, 20), 2e-5)])
def test_hot_path_substage_then_projection(binding, ref, name, size, tol):
    """one substage of the hot path on the GPU gives the predictor u~ (A8); its correction is checked call by call and
    against the oracle's end-to-end long-double correction of the same predictor."""
    from paper_2502_14148_b200 import workloads as W
    B = binding
    cfg = _cfg(W, name, size)
    rg = PU.ref_grid(ref, cfg)
    _, pred, _, gg = PU.run_substage_parity(B, ref, cfg, W.generate_state(cfg), stage=1)
    dt_stage = cfg["dt"] * 8.0 / 15.0
    _call_by_call(B, ref, cfg, pred, dt_stage, tol, hot=True)
    # composed call vs the oracle's chain
    ps = B.ocn_poisson_create(gg)
    st = gg.fields_from_state(pred)
    p = gg.new_field()
    B.ocn_pressure_correction(ps, dt_stage, st, p)
    got = gg.state_from_fields(st)
    want = PU.to64(pred)
    ref.pressure_correction(rg, dt_stage, want)
    for nm in ("u", "v", "w"):
        e, _ = PU.rel_err(rg, got[nm], want[nm])
        assert e <= tol, (nm, e)
    for n in range(len(pred["c"])):                       # tracers are not touched
        assert np.array_equal(got["c"][n], pred["c"][n])


def test_unsupported_and_invalid(binding):
    from paper_2502_14148_b200 import workloads as W
    B = binding
    cfg = W.get_config("C3", size=(48, 40, 12))
    gg = PU.gpu_grid(B, cfg)
    with pytest.raises(B.OcnError) as e:
        B.ocn_poisson_create(gg)
    assert e.value.code == B.OCN_ERR_UNSUPPORTED
    cfg = W.get_config("C1", size=(40, 24, 20))
    gg = PU.gpu_grid(B, cfg)
    st = gg.fields(n_tracers=0)
    p = gg.new_field()
    with pytest.raises(B.OcnError) as e:
        B.ocn_pressure_rhs(gg, 0.0, st, p)
    assert e.value.code == B.OCN_ERR_INVALID
    st.w = None
    with pytest.raises(B.OcnError) as e:
        B.ocn_pressure_rhs(gg, 1.0, st, p)
    assert e.value.code == B.OCN_ERR_INVALID


def test_fullsize_C2_projection_properties(binding):
    """BASELINE size 512x512x256 in the launch configuration bench.py times: div(u^{m+1}) = 0 to rounding and
    lap(p) = rhs, both evaluated by torch slicing on the device arrays (properties that hold at any size)."""
    import torch
    from paper_2502_14148_b200 import workloads as W
    B = binding
    cfg = W.get_config("C2")
    gg = PU.gpu_grid(B, cfg)
    g = cfg["grid"]
    gen = torch.Generator(device="cuda").manual_seed(2025021412)
    st = gg.fields(n_tracers=0)
    for t in (st.u, st.v, st.w):
        gg.interior(t).copy_(0.01 * torch.randn((g["Nz"], g["Ny"], g["Nx"]), device="cuda", dtype=torch.float64, generator=gen))
    gg.interior(st.w)[0] = 0
    ps = B.ocn_poisson_create(gg)
    rhs, p = gg.new_field(), gg.new_field()
    dt = 0.05
    B.ocn_pressure_rhs(gg, dt, st, rhs)
    B.ocn_poisson_solve(ps, rhs, p)
    dx = g["dx"]

    def div(u, v, w):
        wf = torch.cat([w, torch.zeros_like(w[:1])], 0)
        return (torch.roll(u, -1, 2) - u) / dx + (torch.roll(v, -1, 1) - v) / g["dy"] + (wf[1:] - wf[:-1]) / g["dz_uniform"]

    P = gg.interior(p)
    gx = (P - torch.roll(P, 1, 2)) / dx
    gy = (P - torch.roll(P, 1, 1)) / g["dy"]
    gz = torch.zeros_like(P)
    gz[1:] = (P[1:] - P[:-1]) / g["dz_uniform"]
    res = (div(gx, gy, gz) - gg.interior(rhs)).abs().max().item()
    rmax = gg.interior(rhs).abs().max().item()
    assert res <= 1e-11 * rmax, (res, rmax)
    del gx, gy, gz
    B.ocn_pressure_correct(gg, dt, st, p)
    d1 = div(gg.interior(st.u), gg.interior(st.v), gg.interior(st.w)).abs().max().item()
    assert d1 <= 1e-14 * 0.05 / dx * 100, d1
