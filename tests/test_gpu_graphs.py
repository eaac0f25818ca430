"""CUDA-graph replay of the ocn_step* sequences (include/ocn.h ocn_grid_set_graphs; SURVEY 8(f) closing note): the replayed
step is BIT-IDENTICAL to the kernel-by-kernel step, is actually served by graph launches, counts its kernels, and every
argument change (dt, parameters, reference profiles, buffers) selects a different graph.  `-m gpu`."""
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


def _run(B, cfg, graphs, n_steps, entry, p=None, model_opts=None):
    """n_steps full RK3 steps on a side stream; returns (state after, kernel launches counted, graph replays)"""
    import torch
    from paper_2502_14148_b200 import workloads as W
    p = cfg["params"] if p is None else p
    hydro = bool(p["hydrostatic"])
    gg = PU.gpu_grid(B, cfg)
    gg.set_graphs(graphs)
    st = gg.fields_from_state(W.generate_state(cfg))
    G, Gp = PU.new_G(B, gg, cfg), PU.new_G(B, gg, cfg)
    phy = gg.new_field() if hydro else None
    alt = None
    if entry != "step":
        alt = B.Fields(gg.new_field(), gg.new_field(), st.w if hydro else gg.new_field(), [gg.new_field() for _ in st.c])
    kw = {}
    if model_opts == "poisson":
        kw = dict(poisson=B.ocn_poisson_create(gg), p_nh=gg.new_field())
    elif model_opts == "free_surface":
        bt = B.Barotropic(gg)
        B.ocn_barotropic_init(gg, st, bt)
        kw = dict(bt=bt, bt_N=8, bt_weights=W.barotropic_weights(8))
    side = torch.cuda.Stream()
    torch.cuda.synchronize()
    n0 = B.ocn_launch_count()
    cur, oth = st, alt
    with torch.cuda.stream(side):
        for _ in range(n_steps):
            if entry == "step":
                B.ocn_step(gg, p, 3, cfg["dt"], cur, G, Gp, phy)
            elif entry == "fused":
                B.ocn_step_fused(gg, p, 3, cfg["dt"], cur, oth, G, Gp, phy)
                cur, oth = oth, cur               # 3 substages: the result is in the alternate buffers
                G, Gp = Gp, G
            else:
                B.ocn_step_model(gg, p, 3, cfg["dt"], cur, oth, G, Gp, p_hy=phy, **kw)
                cur, oth = oth, cur
                G, Gp = Gp, G
    torch.cuda.synchronize()
    return gg.state_from_fields(cur), B.ocn_launch_count() - n0, gg.graph_replays(), kw


CASES = [("C0", None, "step", None), ("C1", (40, 24, 20), "step", None), ("C1", (40, 24, 20), "fused", None),
         ("C3", (48, 40, 12), "fused", None), ("C4", (40, 24, 20), "fused", None),
         ("C1", (40, 24, 20), "model", "poisson"), ("C3", (48, 40, 12), "model", "free_surface")]


@pytest.mark.parametrize("name,size,entry,opts", CASES)
def test_graph_replay_is_bit_identical(binding, name, size, entry, opts):
    from paper_2502_14148_b200 import workloads as W
    cfg = W.get_config(name, size=size)
    p = cfg["params"]
    if opts == "free_surface":
        p = dict(p, implicit_vertical_diffusion=1)
    n = 6          # the ping-pong entries alternate between two argument sets: each is seen, captured, then replayed
    eager, l0, r0, _ = _run(binding, cfg, False, n, entry, p, opts)
    graph, l1, r1, _ = _run(binding, cfg, True, n, entry, p, opts)
    assert r0 == 0
    assert r1 >= (n - 2 if entry == "step" else n - 4), "the graphs were not used (%d replays)" % r1
    assert l1 == l0, "kernel launches counted differently: eager %d, graphs %d" % (l0, l1)
    for (nm, a), (_, b) in zip(PU.named(eager), PU.named(graph)):
        assert np.array_equal(a, b), "%s %s: %s differs between the eager and the graph-replayed steps" % (name, entry, nm)


def test_every_argument_selects_its_own_graph(binding):
    """changing dt, a parameter, the CONTENTS of the reference profiles or a buffer must not replay a stale graph"""
    import torch
    from paper_2502_14148_b200 import workloads as W
    B = binding
    cfg = W.get_config("C3", size=(48, 40, 12))
    base = cfg["params"]
    variants = [("base", base, cfg["dt"]), ("dt", base, 0.5 * cfg["dt"]), ("nu", dict(base, nu=3e-4), cfg["dt"]),
                ("Tref", dict(base, T_ref=np.asarray(base["T_ref"]) + 0.25), cfg["dt"])]
    results = {}
    for graphs in (False, True):
        gg = PU.gpu_grid(B, cfg)
        gg.set_graphs(graphs)
        G, Gp = PU.new_G(B, gg, cfg), PU.new_G(B, gg, cfg)
        phy = gg.new_field()
        side = torch.cuda.Stream()
        for rnd in range(3):                       # interleave the variants: every one is replayed after the others ran
            for tag, p, dt in variants:
                st = gg.fields_from_state(W.generate_state(cfg))
                if rnd == 0:
                    results.setdefault((tag, "bufs"), (st, B.Fields(gg.new_field(), gg.new_field(), st.w, [gg.new_field() for _ in st.c])))
                st0, alt0 = results[(tag, "bufs")] if graphs else (st, B.Fields(gg.new_field(), gg.new_field(), st.w, [gg.new_field() for _ in st.c]))
                if graphs:                        # same buffers every round so that the key repeats
                    for dst, src in zip([st0.u, st0.v, st0.w] + list(st0.c), [st.u, st.v, st.w] + list(st.c)):
                        dst.copy_(src)
                with torch.cuda.stream(side):
                    side.wait_stream(torch.cuda.current_stream())
                    B.ocn_step_fused(gg, p, 3, dt, st0, alt0, G, Gp, phy)
                torch.cuda.synchronize()
                out = gg.state_from_fields(alt0)
                key = (tag, graphs, rnd)
                results[key] = out
        if graphs:
            assert gg.graph_replays() >= len(variants), gg.graph_replays()
    for tag, _, _ in variants:
        for rnd in range(3):
            for (nm, a), (_, b) in zip(PU.named(results[(tag, False, rnd)]), PU.named(results[(tag, True, rnd)])):
                if nm != "w":
                    assert np.array_equal(a, b), "variant %s round %d: %s differs (stale graph?)" % (tag, rnd, nm)
    # and the variants really differ from each other
    assert not np.array_equal(results[("base", True, 2)]["u"], results[("dt", True, 2)]["u"])
    assert not np.array_equal(results[("base", True, 2)]["u"], results[("Tref", True, 2)]["u"])


def test_a_diagnostic_flag_flipped_after_capture_selects_the_other_kernels(binding):
    """ocn_grid_set_diag is part of the graph key (the library has no environment switch): a hydrostatic ocn_step_fused sequence
    captured with w diagnosed inside the tendency kernel must not be replayed once OCN_DIAG_W_SCAN asks for the ocn_compute_w
    launch — the launch count per step rises by one per substage, state.w is written (ocn_step_writes_w says so beforehand), and
    the prognostic fields stay bit-identical."""
    import torch
    from paper_2502_14148_b200 import workloads as W
    B = binding
    cfg = W.get_config("C3", size=(48, 40, 12))
    p = cfg["params"]
    gg = PU.gpu_grid(B, cfg)
    gg.set_graphs(True)
    G, Gp = PU.new_G(B, gg, cfg), PU.new_G(B, gg, cfg)
    phy = gg.new_field()
    st = gg.fields_from_state(W.generate_state(cfg))
    alt = B.Fields(gg.new_field(), gg.new_field(), st.w, [gg.new_field() for _ in st.c])
    keep = [t.clone() for t in [st.u, st.v] + list(st.c)]
    side = torch.cuda.Stream()
    out, launches, wrote_w = {}, {}, {}
    for tag, mask in (("kernel", 0), ("scan", B.OCN_DIAG_W_SCAN), ("kernel2", 0)):
        gg.set_diag(mask)
        assert B.ocn_step_writes_w(gg, p) == (mask != 0)
        for rnd in range(3):                                # seen, captured, replayed — with identical arguments every time
            for dst, src in zip([st.u, st.v] + list(st.c), keep):
                dst.copy_(src)
            st.w.fill_(123.0)
            torch.cuda.synchronize()
            n0 = B.ocn_launch_count()
            with torch.cuda.stream(side):
                side.wait_stream(torch.cuda.current_stream())
                B.ocn_step_fused(gg, p, 3, cfg["dt"], st, alt, G, Gp, phy)
            torch.cuda.synchronize()
            launches[tag] = B.ocn_launch_count() - n0
        out[tag] = gg.state_from_fields(alt)
        wrote_w[tag] = bool((gg.download(st.w) != 123.0).any())
    assert gg.graph_replays() >= 3
    assert launches["scan"] == launches["kernel"] + 3 and launches["kernel2"] == launches["kernel"], launches
    assert wrote_w == {"kernel": False, "scan": True, "kernel2": False}, wrote_w
    for nm in ("u", "v"):
        assert np.array_equal(out["kernel"][nm], out["scan"][nm]) and np.array_equal(out["kernel"][nm], out["kernel2"][nm])
    with pytest.raises(B.OcnError):
        gg.set_diag(1 << 9)
