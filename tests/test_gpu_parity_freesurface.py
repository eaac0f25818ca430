"""GPU parity of SURVEY 8(f) N4, the split-explicit free surface (A13)-(A21) PAPER.md:857-923, through the C ABI.

P1 teacher-forced: every call (column integrals (A13), slow forcing of (A19), the M forward-backward substeps with their
weighted averages (A18)-(A20), the correction (A21)) is compared element by element with the oracle's long-double evaluation of
THE SAME input arrays; tolerance: the north_star's 1e-12 (fp64) / 2e-5 (fp32) relative to max|field| (a few hundred chained
fp64 operations per point keep the substepper far inside it).  Then the chain on a hot-path predictor, the properties that hold
at any size at the full C3 size, and argument errors."""
import numpy as np
import pytest

from tests import parity_util as PU

pytestmark = pytest.mark.gpu
GRAV = 9.81


@pytest.fixture(scope="module")
def binding():
    import torch
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    from paper_2502_14148_b200 import binding as Bd
    Bd.lib()
    return Bd


def _rel(a, b):
    den = np.abs(b).max()
    return np.abs(np.asarray(a, dtype=np.float64) - b).max() / den if den > 0 else np.abs(a).max()


def _planes_from(ref, rg, bt, B):
    return {k: B.download(getattr(bt, k)).astype(np.float64) for k in ("eta", "U", "V")}


def _setup(B, ref, W, name, size, dtype=None, topology=None):
    cfg = W.get_config(name, size=size)
    if dtype is not None:
        cfg = dict(cfg, dtype=dtype)
    if topology is not None:
        cfg = dict(cfg, grid=dict(cfg["grid"], topology=tuple(topology)))
    return cfg, PU.ref_grid(ref, cfg), PU.gpu_grid(B, cfg)


def _random_bt(B, rg, gg, seed, npdt):
    """physical magnitudes: eta ~ 0.1 m, U ~ H * 0.1 m/s, F ~ H * 1e-5; wall faces of U / V hold 0."""
    r = np.random.default_rng(seed)
    H = rg.metric("dzc").sum()
    bt = B.Barotropic(gg)
    dense = {}
    for key, amp in (("eta", 0.1), ("U", 0.1 * H), ("V", 0.1 * H), ("FU", 1e-5 * H), ("FV", 1e-5 * H)):
        a = np.zeros((rg.nyp, rg.nxp), dtype=npdt)
        a[rg.Hy:rg.Hy + rg.Ny, rg.Hx:rg.Hx + rg.Nx] = (amp * r.standard_normal((rg.Ny, rg.Nx))).astype(npdt)
        if key in ("U", "FU") and rg.topology[0] == 1:
            a[:, rg.Hx] = 0
        if key in ("V", "FV") and rg.topology[1] == 1:
            a[rg.Hy, :] = 0
        dense[key] = a
        bt.upload(getattr(bt, key), a)
    return bt, dense


CASES = [("C3", (48, 40, 12), None), ("C3", (71, 33, 50), None), ("C1", (40, 24, 20), None), ("C3", (48, 40, 12), "f32"),
         ("C1", (16, 9, 70), None),          # Nz > 64: the two-sweep path of the correction kernel
         ("C1", (130, 70, 4), None), ("C3", (150, 64, 6), "f32")]   # planes >= 64 x 32: the S-substeps-per-launch kernel (as (71, 33, 50))


@pytest.mark.parametrize("name,size,dtype", CASES)
def test_column_integrals_and_forcing(binding, ref, name, size, dtype):
    from paper_2502_14148_b200 import workloads as W
    B = binding
    cfg, rg, gg = _setup(B, ref, W, name, size, dtype)
    npdt = np.float64 if cfg["dtype"] == "f64" else np.float32
    tol = PU.TOL[cfg["dtype"]]
    r = np.random.default_rng(2)
    mk = lambda: r.standard_normal(rg.shape).astype(npdt)
    state = {"u": mk(), "v": mk(), "w": None, "c": []}
    Gd = {"u": mk(), "v": mk(), "w": None, "c": []}
    Gpd = {"u": mk(), "v": mk(), "w": None, "c": []}
    st, G, Gp = gg.fields_from_state(state), gg.fields_from_state(Gd), gg.fields_from_state(Gpd)
    bt = B.Barotropic(gg)
    B.ocn_barotropic_init(gg, st, bt)
    want = ref.barotropic_init(rg, PU.to64(state))
    assert _rel(bt.download(bt.U), want["U"]) <= tol and _rel(bt.download(bt.V), want["V"]) <= tol
    for gam, zet, prev in ((8.0 / 15.0, 0.0, None), (1.5, 0.9, (Gp, Gpd))):
        B.ocn_barotropic_forcing(gg, gam, zet, G, None if prev is None else prev[0], bt)
        FU, FV = ref.barotropic_forcing(rg, gam, zet, PU.to64(Gd), None if prev is None else PU.to64(prev[1]))
        assert _rel(bt.download(bt.FU), FU) <= tol and _rel(bt.download(bt.FV), FV) <= tol
    if rg.topology[1] == 1:                                    # wall faces of V hold exactly 0
        assert np.all(bt.download(bt.V)[rg.Hy, rg.Hx:rg.Hx + rg.Nx] == 0)


@pytest.mark.parametrize("name,size,dtype", CASES)
@pytest.mark.parametrize("N", [1, 30])
def test_substeps_teacher_forced(binding, ref, name, size, dtype, N):
    from paper_2502_14148_b200 import workloads as W
    B = binding
    cfg, rg, gg = _setup(B, ref, W, name, size, dtype)
    npdt = np.float64 if cfg["dtype"] == "f64" else np.float32
    bt, dense = _random_bt(B, rg, gg, 5, npdt)
    H = rg.metric("dzc").sum()
    c = np.sqrt(GRAV * H)
    dtau = 0.6 * min(rg.dx, rg.dy) / (np.sqrt(2.0) * c)       # inside the forward-backward limit
    weights = W.barotropic_weights(N) if N > 1 else np.array([1.0])
    assert abs(weights.sum() - 1) < 1e-14 and (N == 1 or N < len(weights) <= 2 * N)
    B.ocn_barotropic_substeps(gg, GRAV, dtau * N, N, weights, bt)
    want = {k: dense[k].astype(np.float64) for k in ("eta", "U", "V")}
    ref.barotropic_substeps(rg, GRAV, dtau * N, N, weights, want, dense["FU"].astype(np.float64), dense["FV"].astype(np.float64))
    tol = PU.TOL[cfg["dtype"]]
    for k in ("eta", "U", "V"):
        got = bt.download(getattr(bt, k))
        assert _rel(got, want[k]) <= tol, (k, _rel(got, want[k]))
        m = np.ones((rg.nyp, rg.nxp), bool)
        m[rg.Hy:rg.Hy + rg.Ny, rg.Hx:rg.Hx + rg.Nx] = False
        assert np.all(got[m] == 0), "halo of %s written" % k
    # the averages differ from the initial state (the test is not vacuous)
    assert _rel(bt.download(bt.eta), dense["eta"].astype(np.float64)) > 1e-3


@pytest.mark.parametrize("name,size,dtype,N", [("C3", (71, 33, 50), None, 30), ("C1", (130, 70, 4), None, 30), ("C3", (150, 64, 6), "f32", 30),
                                               ("C3", (200, 90, 3), None, 7), ("C1", (64, 32, 3), "f32", 2)])
def test_blocked_substeps_are_bit_identical_to_single_substeps(binding, ref, name, size, dtype, N):
    """S substeps per launch on overlapping shared-memory regions (the default for planes >= 64 x 32) == one launch per substep
    (the grid's diagnostic flag OCN_DIAG_BT_SINGLESTEP), bit for bit: same arithmetic per cell, same rounding to the storage type."""
    from paper_2502_14148_b200 import workloads as W
    B = binding
    cfg, rg, gg = _setup(B, ref, W, name, size, dtype)
    npdt = np.float64 if cfg["dtype"] == "f64" else np.float32
    H = rg.metric("dzc").sum()
    dtau = 0.6 * min(rg.dx, rg.dy) / (np.sqrt(2.0) * np.sqrt(GRAV * H))
    weights = W.barotropic_weights(N)
    out = []
    for single in (False, True):
        gg.set_diag(B.OCN_DIAG_BT_SINGLESTEP if single else 0)
        bt, dense = _random_bt(B, rg, gg, 5, npdt)
        B.ocn_barotropic_substeps(gg, GRAV, dtau * N, N, weights, bt)
        out.append({k: bt.download(getattr(bt, k)).copy() for k in ("eta", "U", "V")})
    for k in ("eta", "U", "V"):
        assert np.array_equal(out[0][k], out[1][k]), "%s differs between the blocked and the single-substep kernels" % k
        assert np.isfinite(out[0][k]).all() and np.abs(out[0][k]).max() > 0


@pytest.mark.parametrize("topology", [(1, 1, 1), (1, 0, 1)])
@pytest.mark.parametrize("size", [(48, 40, 6), (100, 50, 4)])      # below / above the 64 x 32 threshold of the blocked kernel
def test_substeps_with_walls_in_x(binding, ref, topology, size):
    """No workload has a wall in x; the substep kernels treat the two axes alike, so both are run on a basin (walls in x and y) and
    on a channel along y, teacher-forced against the oracle."""
    from paper_2502_14148_b200 import workloads as W
    B = binding
    cfg, rg, gg = _setup(B, ref, W, "C3", size, None, topology)
    bt, dense = _random_bt(B, rg, gg, 7, np.float64)
    H = rg.metric("dzc").sum()
    dtau = 0.6 * min(rg.dx, rg.dy) / (np.sqrt(2.0) * np.sqrt(GRAV * H))
    N = 9
    weights = W.barotropic_weights(N)
    B.ocn_barotropic_substeps(gg, GRAV, dtau * N, N, weights, bt)
    want = {k: dense[k].astype(np.float64) for k in ("eta", "U", "V")}
    ref.barotropic_substeps(rg, GRAV, dtau * N, N, weights, want, dense["FU"].astype(np.float64), dense["FV"].astype(np.float64))
    for k in ("eta", "U", "V"):
        got = bt.download(getattr(bt, k))
        assert _rel(got, want[k]) <= PU.TOL["f64"], (k, _rel(got, want[k]))
    assert np.all(bt.download(bt.U)[rg.Hy:rg.Hy + rg.Ny, rg.Hx] == 0)      # the wall face of U stays exactly 0


@pytest.mark.parametrize("name,size,dtype", CASES)
def test_correction_teacher_forced(binding, ref, name, size, dtype):
    from paper_2502_14148_b200 import workloads as W
    B = binding
    cfg, rg, gg = _setup(B, ref, W, name, size, dtype)
    npdt = np.float64 if cfg["dtype"] == "f64" else np.float32
    state = W.generate_state(cfg)
    state = {"u": state["u"].astype(npdt), "v": state["v"].astype(npdt), "w": None, "c": []}
    bt, dense = _random_bt(B, rg, gg, 9, npdt)
    st = gg.fields_from_state(state)
    B.ocn_barotropic_correct(gg, st, bt)
    got = gg.state_from_fields(st)
    want = PU.copy_state(PU.to64(state))
    ref.barotropic_correct(rg, want, {"eta": None, "U": dense["U"].astype(np.float64), "V": dense["V"].astype(np.float64)})
    tol = PU.TOL[cfg["dtype"]]
    for nm in ("u", "v"):
        e, _ = PU.rel_err(rg, got[nm], want[nm])
        assert e <= tol, (nm, e)
        m = np.ones(rg.shape, bool)
        rg.interior(m)[...] = False
        assert np.array_equal(got[nm][m], state[nm][m])


def test_hot_path_chain_C3(binding, ref):
    """a hot-path substage of the hydrostatic config gives the predictor and G; forcing -> substeps -> correction on the GPU,
    each call compared with the oracle applied to the GPU's own inputs."""
    from paper_2502_14148_b200 import workloads as W
    B = binding
    cfg, rg, gg0 = _setup(B, ref, W, "C3", (71, 33, 50))
    p = cfg["params"]
    _, pred, (Gf, G64), gg = PU.run_substage_parity(B, ref, cfg, W.generate_state(cfg), stage=1)
    gam = 8.0 / 15.0
    dt_stage = cfg["dt"] * gam
    st = gg.fields_from_state(pred)
    bt = B.Barotropic(gg)
    B.ocn_barotropic_init(gg, st, bt)
    B.ocn_barotropic_forcing(gg, 1.0, 0.0, Gf, None, bt)               # gamma / (gamma - zeta) = 1 at stage 1
    FU, FV = ref.barotropic_forcing(rg, 1.0, 0.0, G64, None)
    assert _rel(bt.download(bt.FU), FU) <= 1e-12 and _rel(bt.download(bt.FV), FV) <= 1e-12
    start = {k: bt.download(getattr(bt, k)).astype(np.float64) for k in ("eta", "U", "V")}
    FUg, FVg = bt.download(bt.FU).astype(np.float64), bt.download(bt.FV).astype(np.float64)
    N = 20
    weights = W.barotropic_weights(N)
    B.ocn_barotropic_substeps(gg, p["g"], dt_stage, N, weights, bt)
    want = {k: v.copy() for k, v in start.items()}
    ref.barotropic_substeps(rg, p["g"], dt_stage, N, weights, want, FUg, FVg)
    for k in ("eta", "U", "V"):
        assert _rel(bt.download(getattr(bt, k)), want[k]) <= 1e-12, k
    avg = {k: bt.download(getattr(bt, k)).astype(np.float64) for k in ("eta", "U", "V")}
    B.ocn_barotropic_correct(gg, st, bt)
    got = gg.state_from_fields(st)
    wantq = PU.copy_state(PU.to64(pred))
    ref.barotropic_correct(rg, wantq, avg)
    for nm in ("u", "v"):
        e, _ = PU.rel_err(rg, got[nm], wantq[nm])
        assert e <= 1e-12, (nm, e)


def test_fullsize_C3_properties(binding):
    """BASELINE size 1440x600x50: volume conservation of the substepper and sum_k dz u = Ubar after (A21), by torch."""
    import torch
    from paper_2502_14148_b200 import workloads as W
    B = binding
    cfg = W.get_config("C3")
    g = cfg["grid"]
    gg = PU.gpu_grid(B, cfg)
    st = gg.fields_from_state(W.generate_state(cfg, device="cuda", as_numpy=False))
    bt = B.Barotropic(gg)
    B.ocn_barotropic_init(gg, st, bt)
    L = gg.layout
    inner = lambda t: bt.view(t)[L.hy:L.hy + g["Ny"], L.hx:L.hx + g["Nx"]]
    dz = torch.as_tensor(np.asarray(g["dz_c"]), device="cuda")
    U0 = torch.einsum("k,kji->ji", dz, gg.interior(st.u))
    assert (inner(bt.U) - U0).abs().max().item() <= 1e-12 * U0.abs().max().item()
    gen = torch.Generator(device="cuda").manual_seed(7)
    inner(bt.eta).copy_(0.1 * torch.randn((g["Ny"], g["Nx"]), device="cuda", dtype=torch.float64, generator=gen))
    vol0 = inner(bt.eta).sum().item()
    N = 40
    weights = W.barotropic_weights(N)
    B.ocn_barotropic_substeps(gg, 9.81, 400.0, N, weights, bt)
    assert torch.isfinite(inner(bt.eta)).all()
    assert abs(inner(bt.eta).sum().item() - vol0) <= 1e-9 * g["Nx"] * g["Ny"] * 0.1
    B.ocn_barotropic_correct(gg, st, bt)
    U1 = torch.einsum("k,kji->ji", dz, gg.interior(st.u))
    V1 = torch.einsum("k,kji->ji", dz, gg.interior(st.v))
    assert (U1 - inner(bt.U)).abs().max().item() <= 1e-11 * inner(bt.U).abs().max().item()
    assert (V1[1:] - inner(bt.V)[1:]).abs().max().item() <= 1e-11 * inner(bt.V).abs().max().item()
    assert gg.interior(st.v)[:, 0, :].abs().max().item() == 0.0


def test_invalid_arguments(binding):
    from paper_2502_14148_b200 import workloads as W
    B = binding
    cfg = W.get_config("C3", size=(48, 40, 12))
    gg = PU.gpu_grid(B, cfg)
    bt = B.Barotropic(gg)
    for N, M in ((0, 3), (3, 0)):
        with pytest.raises(B.OcnError) as e:
            B.ocn_barotropic_substeps(gg, 9.81, 1.0, N, np.ones(max(M, 0)) if M else np.ones(0), bt)
        assert e.value.code == B.OCN_ERR_INVALID
    with pytest.raises(B.OcnError) as e:
        B.ocn_barotropic_substeps(gg, 9.81, -1.0, 3, np.ones(3) / 3, bt)
    assert e.value.code == B.OCN_ERR_INVALID
    g0 = PU.gpu_grid(B, W.get_config("C0"))
    with pytest.raises(B.OcnError) as e:
        B.ocn_barotropic_correct(g0, g0.fields(n_tracers=0), B.Barotropic(g0))
    assert e.value.code == B.OCN_ERR_INVALID
