"""Shared helpers of the GPU parity tests (and of __graft_entry__.smoke): run one hot-path call on the CUDA
library and the same call on the CPU oracle with THE SAME input arrays (protocol P1, "teacher-forced":
DESIGN.md H3), and compare element by element."""
import numpy as np

TOL = {"f64": 1e-12, "f32": 2e-5}      # BASELINE.json north_star: relative max-norm tolerances


def ref_grid(ref, cfg):
    g = cfg["grid"]
    return ref.RefGrid(g["Nx"], g["Ny"], g["Nz"], g["halo"], g["dx"], g["dy"], g["dz_c"], g["dz_uniform"], g["topology"])


def gpu_grid(B, cfg, kernel=0):
    g = cfg["grid"]
    G = B.ocn_grid_create(g["Nx"], g["Ny"], g["Nz"], g["halo"], g["dx"], g["dy"], g["dz_c"], g["dz_uniform"],
                          g["topology"], cfg["dtype"])
    G.set_kernel(kernel)
    G.set_diag(cfg.get("diag", 0))      # OCN_DIAG_* mask: the reference / fallback kernels stay under test through it
    return G


def to64(state):
    up = lambda a: None if a is None else np.ascontiguousarray(a, dtype=np.float64)
    return {"u": up(state.get("u")), "v": up(state.get("v")), "w": up(state.get("w")), "c": [up(c) for c in state.get("c", [])]}


def copy_state(state):
    cp = lambda a: None if a is None else a.copy()
    return {"u": cp(state.get("u")), "v": cp(state.get("v")), "w": cp(state.get("w")), "c": [cp(c) for c in state.get("c", [])]}


def rel_err(rg, got, want):
    """max_interior |got - want| / max_interior |want|   (SURVEY 8(c) c.7 error metric)"""
    a = rg.interior(np.asarray(got, dtype=np.float64))
    b = rg.interior(np.asarray(want, dtype=np.float64))
    den = np.abs(b).max()
    num = np.abs(a - b).max()
    return num / den if den > 0 else (0.0 if num == 0 else np.inf), den


def named(d):
    out = []
    for k in ("u", "v", "w"):
        if d.get(k) is not None:
            out.append((k, d[k]))
    for n, c in enumerate(d.get("c", [])):
        if c is not None:
            out.append(("c%d" % n, c))
    return out


def new_G(B, G, cfg):
    p = cfg["params"]
    topo = cfg["grid"]["topology"]
    hasw = topo[2] != 2 and not p["hydrostatic"]
    mom = bool(p["momentum_prognostic"])
    # the velocity component along a Flat axis does not exist: no tendency for it
    return G.fields(n_tracers=p["n_tracers"], u=mom and topo[0] != 2, v=mom and topo[1] != 2, w=mom and hasw)


def run_substage_parity(B, ref, cfg, state, kernel=0, stage=1, check_halo_bitwise=True, G_prev_pair=None):
    """One substage on GPU and oracle from the same dense `state` (halos unfilled).  Returns a dict of
    per-field relative errors for tendencies ('G_*') and the updated state ('q_*'), plus both new states."""
    p = cfg["params"]
    rg = ref_grid(ref, cfg)
    gg = gpu_grid(B, cfg, kernel)
    errs = {}
    # ---- GPU: halo fill
    st = gg.fields_from_state(state)
    B.ocn_fill_halos(gg, p, st)
    filled = gg.state_from_fields(st)
    # ---- oracle halo fill on the same input (storage dtype preserved: pure copies => bitwise)
    rs = copy_state(state)
    ref.fill_halos(rg, p, rs)
    for (nm, a), (_, b) in zip(named(filled), named(rs)):
        if nm == "w" and p["hydrostatic"]:
            continue
        if check_halo_bitwise:
            assert np.array_equal(a, b), "halo fill of %s is not bitwise identical" % nm
    phy_gpu = None
    phy_dense = None
    if p["hydrostatic"]:
        B.ocn_compute_w(gg, st)
        w_gpu = gg.download(st.w)
        r64 = to64(filled)
        ref.compute_w(rg, r64)                       # long double scan from the same (filled) u, v
        e, den = rel_err_padded_w(rg, w_gpu, r64["w"])
        errs["w_scan"] = e
        filled["w"] = w_gpu                          # teacher-forcing: downstream oracle calls see the GPU's w
        if p["idx_T"] >= 0 or p["idx_S"] >= 0:
            phy_gpu = gg.new_field()
            B.ocn_compute_phy(gg, p, st, phy_gpu)
            phy_dense = gg.download(phy_gpu)
            pr = ref.compute_phy(rg, p, to64(filled))
            den = np.abs(pr).max()
            errs["p_scan"] = np.abs(phy_dense - pr).max() / den if den > 0 else np.abs(phy_dense).max()
    # ---- tendencies
    Gf = new_G(B, gg, cfg)
    B.ocn_compute_tendencies(gg, p, st, phy_gpu, Gf)
    G_gpu = gg.state_from_fields(Gf)
    in64 = to64(filled)
    G_ref = ref.compute_tendencies(rg, p, in64, None if phy_dense is None else phy_dense.astype(np.float64), eval=0)
    for (nm, a), (_, b) in zip(named(G_gpu), named(G_ref)):
        errs["G_" + nm], _ = rel_err(rg, a, b)
    # ---- RK3 substage with the GPU's tendencies as input on both sides
    if G_prev_pair is None:
        Gp_f, Gp_ref = None, None
    else:
        Gp_f, Gp_ref = G_prev_pair
    B.ocn_rk3_substage(gg, p, stage, cfg["dt"], st, Gf, Gp_f)
    new_gpu = gg.state_from_fields(st)
    old = {nm: np.array(a, copy=True) for nm, a in named(filled)}      # to64 does not copy float64 arrays: keep q_old for the increment check
    new_ref = to64(filled)
    G64 = to64(G_gpu)
    ref.rk3_substage(rg, p, stage, cfg["dt"], new_ref, G64, Gp_ref, eval=0)
    for (nm, a), (_, b) in zip(named(new_gpu), named(new_ref)):
        errs["q_" + nm], _ = rel_err(rg, a, b)
    # ---- the INCREMENT of (A4): dq = q_new - q_old on both sides from the same q_old (the filled state)
    for (nm, a), (_, b) in zip(named(new_gpu), named(new_ref)):
        if nm == "w" and p["hydrostatic"]:
            continue
        errs["dq_" + nm], errs["_dqtol_" + nm] = increment_err(rg, cfg["dtype"], old[nm], a, b)
    return errs, new_gpu, (Gf, G64), gg


EPS = {"f64": 2.0 ** -52, "f32": 2.0 ** -23}


def increment_err(rg, dtype, q_old, q_gpu, q_ref):
    """(error of the substage increment relative to the increment, its tolerance).
    error = max|(q_gpu - q_old) - (q_ref - q_old)| / max|q_ref - q_old| over the interior.  q_old is the same array on both
    sides, so this is the q-error rescaled by max|q| / max|dq| (T ~ 20, S ~ 35 against increments of ~1e-5): a wrong gamma, zeta
    or dt in a tracer path shows up at O(1) here instead of hiding behind the size of the field.  Tolerance: the substage stores
    q_new in the field's dtype, so each side carries one rounding of up to ulp(q)/2 that no arithmetic can avoid (the oracle returns
    its long-double result rounded to double; a float32 state is rounded again by the GPU's store): the floor is
    eps_dtype * max|q| / max|dq|, and the tolerance is the north_star's TOL plus twice that floor."""
    o = rg.interior(np.asarray(q_old, dtype=np.float64))
    a = rg.interior(np.asarray(q_gpu, dtype=np.float64))
    b = rg.interior(np.asarray(q_ref, dtype=np.float64))
    dq = np.abs(b - o).max()
    qmax = max(np.abs(b).max(), np.abs(o).max())
    if dq == 0:
        return (0.0 if np.array_equal(a, b) else np.inf), 0.0
    return np.abs(a - b).max() / dq, TOL[dtype] + 2.0 * EPS[dtype] * qmax / dq


def rel_err_padded_w(rg, got, want):
    """w from the scan is defined on levels 1..Nz+1 and on all columns but the last in x and y."""
    a = np.asarray(got, dtype=np.float64)[rg.Hz:rg.Hz + rg.Nz + 1, :rg.nyp - 1 if rg.Hy else rg.nyp, :rg.nxp - 1 if rg.Hx else rg.nxp]
    b = np.asarray(want, dtype=np.float64)[rg.Hz:rg.Hz + rg.Nz + 1, :rg.nyp - 1 if rg.Hy else rg.nyp, :rg.nxp - 1 if rg.Hx else rg.nxp]
    den = np.abs(b).max()
    num = np.abs(a - b).max()
    return (num / den if den > 0 else num), den


def assert_errs(errs, dtype, what=""):
    tol = TOL[dtype]
    # "dq_X" (increment of the substage) carries its own tolerance "_dqtol_X" (increment_err); everything else the north_star's
    bad = {k: v for k, v in errs.items() if not k.startswith("_") and not (v <= errs.get("_dqtol_" + k[3:], tol) if k.startswith("dq_") else v <= tol)}
    assert not bad, "%s parity beyond %.0e: %s (all: %s)" % (what, tol, bad, errs)
