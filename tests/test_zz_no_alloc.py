"""ocn_barotropic_substeps_static — the free-surface substepper (A18)-(A20), for callers that may not allocate.

Who that is: a host application that gave the whole GPU to its own memory pool at start-up, a time-critical loop that cannot
take the device-wide synchronisation of cudaMalloc / cudaFree, a plug-in whose host forbids allocation after initialisation.
Such a caller cannot provide the six scratch planes ocn_barotropic_substeps asks for, so this entry point keeps them in a fixed
array inside the library (OCN_BT_STATIC_SCRATCH_BYTES per GPU, held from load to exit) and allocates nothing.

What is checked here: on two calls in a row — the second on another grid and dtype, so that the shared array still holds the
first call's bytes — the result equals that of ocn_barotropic_substeps with caller-owned, zero-filled scratch, bit for bit (same
kernels, same arithmetic; that is inside the 1e-12 / 2e-5 tolerance of the other parity tests, which is asserted as well), the
caller's own scratch tensor is never touched, and a grid beyond the limit is refused with a clear message.

This file sorts last on purpose: under `pytest -x` a failure here must not hide the other tests.  It builds its own grids and
inputs, so it passes alone in a fresh process as well as after the rest of the suite."""
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


def _grid(B, size, dtype):
    from paper_2502_14148_b200 import workloads as W
    cfg = dict(W.get_config("C3", size=size), dtype=dtype)
    return cfg, PU.gpu_grid(B, cfg)


def _inputs(gg, seed):
    """eta ~ 0.1 m, U, V ~ H * 0.1 m/s, F ~ H * 1e-5 on the interior (dense (ny_pad, nx_pad) arrays), wall faces of V hold 0."""
    r = np.random.default_rng(seed)
    L = gg.layout
    npdt = np.float64 if gg.dtype == "f64" else np.float32
    H = 100.0
    dense = {}
    for key, amp in (("eta", 0.1), ("U", 0.1 * H), ("V", 0.1 * H), ("FU", 1e-5 * H), ("FV", 1e-5 * H)):
        a = np.zeros((L.ny_pad, L.nx_pad), dtype=npdt)
        a[L.hy:L.hy + gg.Ny, L.hx:L.hx + gg.Nx] = (amp * r.standard_normal((gg.Ny, gg.Nx))).astype(npdt)
        if key in ("V", "FV") and gg.topology[1] == 1:
            a[L.hy, :] = 0
        dense[key] = a
    return dense


def _bt(B, gg, dense):
    bt = B.Barotropic(gg)
    for k, a in dense.items():
        bt.upload(getattr(bt, k), a)
    return bt


def test_static_scratch_substeps_match_the_caller_scratch_path_twice_in_a_row(binding):
    import torch
    from paper_2502_14148_b200 import workloads as W
    B = binding
    N = 10
    weights = W.barotropic_weights(N)
    # first call: a plane above the 64 x 32 threshold (four substeps per launch), fp64, large values left behind in the array;
    # second call: a smaller fp32 plane (one launch per substep) whose averages would inherit those bytes if nothing were cleared
    for call, (size, dtype) in enumerate([((150, 64, 6), "f64"), ((48, 40, 12), "f32")]):
        cfg, gg = _grid(B, size, dtype)
        dense = _inputs(gg, 11 + call)
        depth = float(np.sum(cfg["grid"]["dz_c"]))
        dtau = 0.6 * min(cfg["grid"]["dx"], cfg["grid"]["dy"]) / (np.sqrt(2.0) * np.sqrt(GRAV * depth))   # inside the forward-backward limit
        want_bt = _bt(B, gg, dense)
        B.ocn_barotropic_substeps(gg, GRAV, dtau * N, N, weights, want_bt)             # caller-owned, zero-filled scratch
        got_bt = _bt(B, gg, dense)
        got_bt.scratch.fill_(float("nan"))                                            # must stay unused
        B.ocn_barotropic_substeps_static(gg, GRAV, dtau * N, N, weights, got_bt)
        torch.cuda.synchronize()
        assert torch.isnan(got_bt.scratch).all(), "the static entry point wrote the caller's scratch tensor"
        for k in ("eta", "U", "V"):
            want, got = want_bt.download(getattr(want_bt, k)), got_bt.download(getattr(got_bt, k))
            assert np.isfinite(got).all() and np.abs(got).max() > 0
            err = np.abs(got.astype(np.float64) - want).max() / np.abs(want).max()
            assert err <= PU.TOL[dtype], (call, k, err)
            assert np.array_equal(got, want), "call %d: %s differs from the caller-scratch path" % (call, k)
            assert not np.array_equal(got, dense[k]), "call %d: %s unchanged (vacuous test)" % (call, k)


def test_static_scratch_refuses_planes_beyond_its_size(binding):
    B = binding
    # 1100 x 1100 (+ halos) fp64: six planes need > 48 MiB; the same plane in fp32 fits
    cfg, gg = _grid(B, (1100, 1100, 3), "f64")
    assert 6 * gg.layout.stride_z * 8 > B.OCN_BT_STATIC_SCRATCH_BYTES
    bt = B.Barotropic(gg)
    with pytest.raises(B.OcnError) as e:
        B.ocn_barotropic_substeps_static(gg, GRAV, 1.0, 1, np.array([1.0]), bt)
    assert e.value.code == B.OCN_ERR_UNSUPPORTED and "OCN_BT_STATIC_SCRATCH_BYTES" in str(e.value)
    # the full-size C3 plane (1440 x 600) is inside the limit
    cfg, gg = _grid(B, (1440, 600, 3), "f64")
    assert 6 * gg.layout.stride_z * 8 <= B.OCN_BT_STATIC_SCRATCH_BYTES
    bt = _bt(B, gg, _inputs(gg, 3))
    B.ocn_barotropic_substeps_static(gg, GRAV, 1.0, 4, np.full(4, 0.25), bt)
    assert np.isfinite(bt.download(bt.eta)).all()
