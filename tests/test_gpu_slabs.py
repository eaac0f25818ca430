"""Multi-GPU y-slabs on ONE device: R slabs of the same grid live on cuda:0 as R local ocn_grids marked
ocn_grid_set_external_halo(1); per substage each slab runs ocn_fill_halos (x, z halos), the slabs swap their H outermost rows
through libocn's pack / unpack kernels (the transport is a device copy here, NCCL send/recv between processes in
`slab.YSlabs.exchange`), then ocn_tendencies_rk3.  After a full RK3 step the slabs' interiors must equal the single-grid run
BIT FOR BIT.  The ranks are emulated sequentially: no kernel waits for another (B200_PROFILING.md)."""
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


@pytest.mark.parametrize("name,size,R,order,beta", [("C1", (40, 24, 20), 2, 5, 0.0), ("C1", (67, 35, 9), 3, 5, 0.0), ("C4", (40, 24, 20), 2, 5, 0.0),
                                                    ("C1", (40, 30, 12), 2, 9, 0.0),
                                                    # beta-plane: f varies by a factor 5 over the rows; the kernels see LOCAL row indices, so every
                                                    # slab is given its own y-origin (YSlabs.local_params); dy = 1 keeps the shifted y exact
                                                    ("C1", (40, 24, 20), 2, 5, 2e-5), ("C1", (67, 35, 9), 3, 5, 2e-5), ("C1", (40, 30, 12), 2, 9, 2e-5)])
def test_slabs_reproduce_the_single_grid_step(binding, name, size, R, order, beta):
    import torch
    from paper_2502_14148_b200 import workloads as W
    from paper_2502_14148_b200.slab import YSlabs
    B = binding
    cfg = W.get_config(name, size=size, weno_order=order)
    p, g = cfg["params"], cfg["grid"]
    if beta:
        p = dict(p, beta_coriolis=beta, y0=2.0)
        cfg = dict(cfg, params=p)
    Hh = g["halo"]
    dt = cfg["dt"]
    state = W.generate_state(cfg)
    fused = order == 5
    # ---- single grid
    gg = PU.gpu_grid(B, cfg)
    st = gg.fields_from_state(state)
    G, Gp = PU.new_G(B, gg, cfg), PU.new_G(B, gg, cfg)
    if fused:
        alt = gg.fields(n_tracers=p["n_tracers"])
        B.ocn_step_fused(gg, p, 3, dt, st, alt, G, Gp, None)
        want = gg.state_from_fields(alt)
    else:
        B.ocn_step(gg, p, 3, dt, st, G, Gp, None)
        want = gg.state_from_fields(st)
    # ---- R slabs on the same device
    slabs = []
    for r in range(R):
        sl = YSlabs(g["Ny"], Hh, R, r)
        lcfg = dict(cfg, grid=dict(g, Ny=sl.ny_local))
        lg = PU.gpu_grid(B, lcfg)
        lg.set_external_halo(1, True)
        rows = slice(Hh + sl.j0, Hh + sl.j0 + sl.ny_local)
        cut = lambda a: None if a is None else np.ascontiguousarray(np.concatenate(
            [np.zeros_like(a[:, :Hh, :]), a[:, rows, :], np.zeros_like(a[:, :Hh, :])], axis=1))
        lstate = {"u": cut(state["u"]), "v": cut(state["v"]), "w": cut(state["w"]), "c": [cut(c) for c in state["c"]]}
        cur = lg.fields_from_state(lstate)
        slabs.append(dict(sl=sl, cfg=lcfg, g=lg, cur=cur, p=sl.local_params(p, g["dy"]), alt=lg.fields(n_tracers=p["n_tracers"]), G=PU.new_G(B, lg, lcfg),
                          Gp=PU.new_G(B, lg, lcfg), bufs=sl.make_buffers(B, lg, p)))
    for m in (1, 2, 3):
        for s in slabs:
            B.ocn_fill_halos(s["g"], p, s["cur"])
            B.ocn_halo_pack_y(s["g"], p, s["cur"], 0, s["bufs"]["send_lo"])
            B.ocn_halo_pack_y(s["g"], p, s["cur"], 1, s["bufs"]["send_hi"])
        for s in slabs:                                   # the transport: what NCCL send/recv does between processes
            s["bufs"]["recv_lo"].copy_(slabs[s["sl"].south]["bufs"]["send_hi"])
            s["bufs"]["recv_hi"].copy_(slabs[s["sl"].north]["bufs"]["send_lo"])
        for s in slabs:
            B.ocn_halo_unpack_y(s["g"], p, s["cur"], 0, s["bufs"]["recv_lo"])
            B.ocn_halo_unpack_y(s["g"], p, s["cur"], 1, s["bufs"]["recv_hi"])
            if fused:
                B.ocn_tendencies_rk3(s["g"], s["p"], m, dt, s["cur"], None, s["G"], None if m == 1 else s["Gp"], s["alt"])
                s["cur"], s["alt"] = s["alt"], s["cur"]
            else:
                B.ocn_compute_tendencies(s["g"], s["p"], s["cur"], None, s["G"])
                B.ocn_rk3_substage(s["g"], p, m, dt, s["cur"], s["G"], None if m == 1 else s["Gp"])
            s["G"], s["Gp"] = s["Gp"], s["G"]
    torch.cuda.synchronize()
    rg = PU.ref_grid(binding and __import__("oracle.ocnref", fromlist=["x"]), cfg)
    for s in slabs:
        got = s["g"].state_from_fields(s["cur"])
        sl = s["sl"]
        for (nm, a), (_, b) in zip(PU.named(got), PU.named(want)):
            ai = a[Hh:a.shape[0] - Hh, Hh:Hh + sl.ny_local, Hh:a.shape[2] - Hh]
            bi = rg.interior(b)[:, sl.local_slice(), :]
            assert np.array_equal(ai, bi), "%s slab %d: %s differs from the single-grid step" % (name, sl.rank, nm)


def test_external_halo_rules(binding):
    from paper_2502_14148_b200 import workloads as W
    B = binding
    c3 = W.get_config("C3", size=(48, 40, 12))           # Bounded y: a wall on a slab boundary is not built
    g3 = PU.gpu_grid(B, c3)
    with pytest.raises(B.OcnError) as e:
        g3.set_external_halo(1, True)
    assert e.value.code == B.OCN_ERR_UNSUPPORTED
    c1 = W.get_config("C1", size=(40, 24, 20))
    g1 = PU.gpu_grid(B, c1)
    with pytest.raises(B.OcnError) as e:                 # never split z (the column scans stay local)
        g1.set_external_halo(2, True)
    assert e.value.code == B.OCN_ERR_UNSUPPORTED
    # external y halos are left alone by ocn_fill_halos, x and z halos are filled
    import torch
    g1.set_external_halo(1, True)
    st = g1.fields_from_state(W.generate_state(c1))
    for t in st.all():
        v = g1.view(t)
        v[:, :3, :] = 7.0
        v[:, -3:, :] = 7.0
    B.ocn_fill_halos(g1, c1["params"], st)
    torch.cuda.synchronize()
    for t in st.all():
        v = g1.view(t)
        assert bool((v[:, :3, :] == 7.0).all()) and bool((v[:, -3:, :] == 7.0).all())
    u = g1.view(st.c[0])
    assert bool((u[3:-3, 3:-3, :3] == u[3:-3, 3:-3, -6:-3]).all())          # periodic x halo filled
    # entry points with no exchange hook, and solvers that would wrap y inside the slab, refuse a slab grid
    p1 = c1["params"]
    alt, G, Gp = g1.fields(n_tracers=2), PU.new_G(B, g1, c1), PU.new_G(B, g1, c1)
    bt = B.Barotropic(g1)
    for call in (lambda: B.ocn_step(g1, p1, 3, c1["dt"], st, G, Gp, None),
                 lambda: B.ocn_step_fused(g1, p1, 3, c1["dt"], st, alt, G, Gp, None),
                 lambda: B.ocn_step_model(g1, p1, 3, c1["dt"], st, alt, G, Gp),
                 lambda: B.ocn_poisson_create(g1),
                 lambda: B.ocn_barotropic_substeps(g1, 9.81, 1.0, 1, np.array([1.0]), bt)):
        with pytest.raises(B.OcnError) as e:
            call()
        assert e.value.code == B.OCN_ERR_UNSUPPORTED and "slab" in str(e.value), str(e.value)
    g1.set_external_halo(1, False)                                            # and accept it again once it is a whole grid
    B.ocn_step_fused(g1, p1, 3, c1["dt"], st, alt, G, Gp, None)
    torch.cuda.synchronize()
