"""Full-size parity (BASELINE.json sizes C2, C3, C4) in the launch configuration bench.py times: one substage
{ocn_fill_halos, [ocn_compute_w, ocn_compute_phy], ocn_tendencies_rk3} on the full grid, then SAMPLED SUB-BOXES are
checked element by element against the oracle.

A sub-box is a window of (i, j) columns over the FULL depth, cut out of the GPU's halo-filled state together with
its 3-cell rim.  The oracle evaluates the tendencies of the window from exactly those arrays (teacher-forced,
DESIGN.md 7 P1): in x / y the window's rim plays the part of the halo (oracle topology Periodic, no fill), in z the
window holds the real walls, so every value the oracle returns is the value of the discrete formulas at that cell
of the full grid.  The error metric and tolerances are the north_star's (relative max-norm over the window,
1e-12 fp64 / 2e-5 fp32); G is compared first, then the state written by the fused substage (stage 2, so G_prev is
exercised) against the oracle's (A4) applied to the GPU's own G.
"""
import numpy as np
import pytest

from tests import parity_util as PU

pytestmark = pytest.mark.gpu

H = 3


@pytest.fixture(scope="module")
def binding():
    import torch
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    from paper_2502_14148_b200 import binding as Bd
    Bd.lib()
    return Bd


def _window(gg, t, i0, j0, nx, ny):
    """dense (nz_pad, ny+2H, nx+2H) float64 copy of the window of interior cells i0..i0+nx-1, j0..j0+ny-1 (1-based)
    plus its rim, from layout buffer t."""
    v = gg.view(t)
    return v[:, j0 - 1:j0 - 1 + ny + 2 * H, i0 - 1:i0 - 1 + nx + 2 * H].to("cpu").double().numpy().copy()


def _boxes(cfg):
    g = cfg["grid"]
    Nx, Ny = g["Nx"], g["Ny"]
    nx, ny = 37, 13                                   # spans two x-tiles (31) and three y-tiles (6) of the fused kernel
    out = [(1, 1), (Nx - nx + 1, Ny - ny + 1), (Nx // 2 - 5, Ny // 3), (29, Ny - ny - 40), (Nx - nx - 17, 5)]
    return [(i, j, nx, ny) for (i, j) in out]


@pytest.mark.parametrize("name", ["C2", "C3", "C4"])
def test_fullsize_sampled_boxes(binding, ref, name):
    import torch
    from paper_2502_14148_b200 import workloads as W
    B = binding
    cfg = W.get_config(name)
    p, g = cfg["params"], cfg["grid"]
    hydro = bool(p["hydrostatic"])
    gg = PU.gpu_grid(B, cfg)
    st = gg.fields_from_state(W.generate_state(cfg, device="cuda", as_numpy=False))
    torch.cuda.empty_cache()
    alt = B.Fields(gg.new_field(), gg.new_field(), st.w if hydro else gg.new_field(), [gg.new_field() for _ in st.c])
    G, Gp = PU.new_G(B, gg, cfg), PU.new_G(B, gg, cfg)
    phy = gg.new_field() if hydro else None
    dt = cfg["dt"]
    # stage 1 produces a G_prev and a new state; the checked substage is stage 2 from that state
    B.ocn_fill_halos(gg, p, st)
    if hydro:
        B.ocn_compute_w(gg, st); B.ocn_compute_phy(gg, p, st, phy)
    B.ocn_tendencies_rk3(gg, p, 1, dt, st, phy, Gp, None, alt)
    cur, nxt = alt, st
    B.ocn_fill_halos(gg, p, cur)
    if hydro:
        B.ocn_compute_w(gg, cur); B.ocn_compute_phy(gg, p, cur, phy)
    B.ocn_tendencies_rk3(gg, p, 2, dt, cur, phy, G, Gp, nxt)
    torch.cuda.synchronize()
    tol = PU.TOL[cfg["dtype"]]
    # global scale of every tendency (the north_star's max-norm is over the whole interior)
    names = ["u", "v"] + ([] if hydro else ["w"]) + ["c%d" % n for n in range(p["n_tracers"])]
    fld = lambda F, nm: F.c[int(nm[1:])] if nm.startswith("c") else getattr(F, nm)
    gmax = {nm: float(gg.interior(fld(G, nm)).abs().max()) for nm in names}
    qmax = {nm: float(gg.interior(fld(nxt, nm)).abs().max()) for nm in names}
    worst = {}
    for (i0, j0, nx, ny) in _boxes(cfg):
        south_wall = g["topology"][1] == 1 and j0 == 1
        topo = (0, 1 if south_wall else 0, g["topology"][2])
        pb = dict(p)
        pb["y0"] = p["y0"] - (j0 - 1) * g["dy"]          # f = f0 + beta (y - y0), y measured from the window's south face
        rg = ref.RefGrid(nx, ny, g["Nz"], H, g["dx"], g["dy"], g["dz_c"], g["dz_uniform"], topo)
        win = lambda t: None if t is None else _window(gg, t, i0, j0, nx, ny)
        s_in = {"u": win(cur.u), "v": win(cur.v), "w": win(cur.w), "c": [win(t) for t in cur.c]}
        G_ref = ref.compute_tendencies(rg, pb, s_in, win(phy) if hydro else None, eval=0)
        G_gpu = {"u": win(G.u), "v": win(G.v), "w": win(G.w), "c": [win(t) for t in G.c]}
        Gp_gpu = {"u": win(Gp.u), "v": win(Gp.v), "w": win(Gp.w), "c": [win(t) for t in Gp.c]}
        for (nm, a), (_, b) in zip(PU.named(G_gpu), PU.named(G_ref)):
            e = np.abs(rg.interior(a) - rg.interior(b)).max() / gmax[nm]
            worst["G_" + nm] = max(worst.get("G_" + nm, 0.0), e)
        q_ref = {k: (None if v is None else v.copy()) for k, v in s_in.items() if k != "c"}
        q_ref["c"] = [c.copy() for c in s_in["c"]]
        ref.rk3_substage(rg, pb, 2, dt, q_ref, G_gpu, Gp_gpu, eval=0)
        q_gpu = {"u": win(nxt.u), "v": win(nxt.v), "w": win(nxt.w), "c": [win(t) for t in nxt.c]}
        for (nm, a), (_, b) in zip(PU.named(q_gpu), PU.named(q_ref)):
            if nm == "w" and hydro:
                continue
            e = np.abs(rg.interior(a) - rg.interior(b)).max() / qmax[nm]
            worst["q_" + nm] = max(worst.get("q_" + nm, 0.0), e)
    print("%s full size: worst relative errors %s" % (name, {k: "%.2e" % v for k, v in worst.items()}))
    PU.assert_errs(worst, cfg["dtype"], "%s full size" % name)
    assert tol > 0


@pytest.mark.parametrize("order", [7, 9])
def test_fullsize_c2_weno9_sampled_boxes(binding, ref, order):
    """SURVEY 8(f) N1 at the benched size: `bench.py --weno-order 7|9` runs {ocn_fill_halos, ocn_tendencies_rk3} on the TMA-staged
    marching kernel (grid (17, 64, 3) at C2).  Same sampled-window protocol as above with halo 4 / 5: stage 1 makes a G_prev,
    stage 2 is checked through the two-call path (G against the oracle's WENO7/9 tendencies of the window, the state against (A4)),
    and the fused call the bench times must reproduce that path bit for bit over the whole grid."""
    import torch
    from paper_2502_14148_b200 import workloads as W
    B = binding
    cfg = W.get_config("C2", weno_order=order)
    p, g = cfg["params"], cfg["grid"]
    Hh = g["halo"]
    assert Hh == (order + 1) // 2
    gg = PU.gpu_grid(B, cfg)
    st = gg.fields_from_state(W.generate_state(cfg, device="cuda", as_numpy=False))
    torch.cuda.empty_cache()
    G, Gp = PU.new_G(B, gg, cfg), PU.new_G(B, gg, cfg)
    dt = cfg["dt"]
    B.ocn_fill_halos(gg, p, st)
    B.ocn_compute_tendencies(gg, p, st, None, Gp)
    B.ocn_rk3_substage(gg, p, 1, dt, st, Gp, None)
    B.ocn_fill_halos(gg, p, st)
    B.ocn_compute_tendencies(gg, p, st, None, G)
    torch.cuda.synchronize()

    def window(t, i0, j0, nx, ny):
        v = gg.view(t)
        return v[:, j0 - 1:j0 - 1 + ny + 2 * Hh, i0 - 1:i0 - 1 + nx + 2 * Hh].to("cpu").double().numpy().copy()
    names = ["u", "v", "w", "c0", "c1"]
    fld = lambda F, nm: F.c[int(nm[1:])] if nm.startswith("c") else getattr(F, nm)
    gmax = {nm: float(gg.interior(fld(G, nm)).abs().max()) for nm in names}
    boxes = _boxes(cfg)
    s_ins = []
    for (i0, j0, nx, ny) in boxes:          # the substage updates the state in place: cut the input windows first
        win = lambda t: window(t, i0, j0, nx, ny)
        s_ins.append({"u": win(st.u), "v": win(st.v), "w": win(st.w), "c": [win(t) for t in st.c]})
    # the fused call of the bench (tendencies + substage in one pass, ping-pong state) on the same inputs, before they are updated
    G2, alt = PU.new_G(B, gg, cfg), gg.fields(n_tracers=p["n_tracers"])
    B.ocn_tendencies_rk3(gg, p, 2, dt, st, None, G2, Gp, alt)
    B.ocn_rk3_substage(gg, p, 2, dt, st, G, Gp)
    torch.cuda.synchronize()
    for nm in names:
        assert torch.equal(gg.interior(fld(G2, nm)), gg.interior(fld(G, nm))), "WENO%d full size: fused G_%s differs from the two-call path" % (order, nm)
        assert torch.equal(gg.interior(fld(alt, nm)), gg.interior(fld(st, nm))), "WENO%d full size: fused state %s differs from the two-call path" % (order, nm)
    del G2, alt
    torch.cuda.empty_cache()
    qmax = {nm: float(gg.interior(fld(st, nm)).abs().max()) for nm in names}
    worst = {}
    for (i0, j0, nx, ny), s_in in zip(boxes, s_ins):
        rg = ref.RefGrid(nx, ny, g["Nz"], Hh, g["dx"], g["dy"], g["dz_c"], g["dz_uniform"], (0, 0, g["topology"][2]))
        win = lambda t: window(t, i0, j0, nx, ny)
        G_ref = ref.compute_tendencies(rg, p, s_in, None, eval=0)
        G_gpu = {"u": win(G.u), "v": win(G.v), "w": win(G.w), "c": [win(t) for t in G.c]}
        Gp_gpu = {"u": win(Gp.u), "v": win(Gp.v), "w": win(Gp.w), "c": [win(t) for t in Gp.c]}
        for (nm, a), (_, b) in zip(PU.named(G_gpu), PU.named(G_ref)):
            worst["G_" + nm] = max(worst.get("G_" + nm, 0.0), np.abs(rg.interior(a) - rg.interior(b)).max() / gmax[nm])
        q_ref = {"u": s_in["u"].copy(), "v": s_in["v"].copy(), "w": s_in["w"].copy(), "c": [c.copy() for c in s_in["c"]]}
        ref.rk3_substage(rg, p, 2, dt, q_ref, G_gpu, Gp_gpu, eval=0)
        q_gpu = {"u": win(st.u), "v": win(st.v), "w": win(st.w), "c": [win(t) for t in st.c]}
        for (nm, a), (_, b) in zip(PU.named(q_gpu), PU.named(q_ref)):
            worst["q_" + nm] = max(worst.get("q_" + nm, 0.0), np.abs(rg.interior(a) - rg.interior(b)).max() / qmax[nm])
    print("C2 WENO%d full size: worst relative errors %s" % (order, {k: "%.2e" % v for k, v in worst.items()}))
    PU.assert_errs(worst, cfg["dtype"], "C2 WENO%d full size" % order)
