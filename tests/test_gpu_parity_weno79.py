"""GPU parity of the WENO7 / WENO9 path: ocn_fill_halos (halo 4, 5), ocn_compute_tendencies through the
general high-order kernel (tend_hiorder.cu), ocn_rk3_substage — teacher-forced against the long-double oracle, same
tolerances as the WENO5 path (1e-12 fp64, 2e-5 fp32; halo fill bitwise).  Run with `pytest -m gpu` on the B200 box."""
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


@pytest.fixture(scope="module")
def W():
    from paper_2502_14148_b200 import workloads
    return workloads


def _three_substages(binding, ref, cfg, state, kernel=0):
    """kernel 0: the marching kernel on 3-D grids (every face flux once); kernel 1: the per-cell high-order kernel"""
    prev = None
    for stage in (1, 2, 3):
        errs, new_gpu, (Gf, G64), gg = PU.run_substage_parity(binding, ref, cfg, state, kernel=kernel, stage=stage, G_prev_pair=prev)
        PU.assert_errs(errs, cfg["dtype"], "%s WENO%d stage %d" % (cfg["name"], cfg["weno_order"], stage))
        prev = (Gf, G64)
        state = new_gpu
    return state


@pytest.mark.parametrize("order", [7, 9])
def test_c0_weno79(binding, ref, W, order):
    cfg = W.get_config("C0", weno_order=order)
    _three_substages(binding, ref, cfg, W.generate_state(cfg))


@pytest.mark.parametrize("kernel", [0, 1])
@pytest.mark.parametrize("order", [7, 9])
@pytest.mark.parametrize("size", [(40, 24, 20), (67, 35, 9)])
def test_c1_weno79(binding, ref, W, order, size, kernel):
    cfg = W.get_config("C1", size=size, weno_order=order)
    _three_substages(binding, ref, cfg, W.generate_state(cfg), kernel)


@pytest.mark.parametrize("order", [7, 9])
def test_c2_spectrum_weno79(binding, ref, W, order):
    cfg = W.get_config("C2", size=(64, 48, 32), weno_order=order)
    _three_substages(binding, ref, cfg, W.generate_state(cfg))


@pytest.mark.parametrize("kernel", [0, 1])
@pytest.mark.parametrize("order", [7, 9])
@pytest.mark.parametrize("size", [(48, 40, 12), (71, 33, 50)])
def test_c3_hydrostatic_weno79(binding, ref, W, order, size, kernel):
    cfg = W.get_config("C3", size=size, weno_order=order)
    _three_substages(binding, ref, cfg, W.generate_state(cfg), kernel)


@pytest.mark.parametrize("kernel", [0, 1])
@pytest.mark.parametrize("order", [7, 9])
def test_c4_fp32_weno79(binding, ref, W, order, kernel):
    cfg = W.get_config("C4", size=(40, 24, 20), weno_order=order)
    _three_substages(binding, ref, cfg, W.generate_state(cfg), kernel)


@pytest.mark.parametrize("order", [7, 9])
@pytest.mark.parametrize("name,size", [("C1", (67, 35, 9)), ("C3", (48, 40, 12)), ("C4", (40, 24, 20))])
def test_unstaged_march_kernel_weno79(binding, ref, W, monkeypatch, name, size, order):
    """The global-load marching kernel (the fallback of the TMA-staged one: more than 3 tracers, tiles that do not fit two
    blocks per SM) stays under test through the library's diagnostic switch OCN_HI_NOSTAGE (read at every launch)."""
    monkeypatch.setenv("OCN_HI_NOSTAGE", "1")
    cfg = W.get_config(name, size=size, weno_order=order)
    _three_substages(binding, ref, cfg, W.generate_state(cfg))


def test_c1_full_weno9(binding, ref, W):
    cfg = W.get_config("C1", weno_order=9)
    errs, *_ = PU.run_substage_parity(binding, ref, cfg, W.generate_state(cfg), kernel=0, stage=1)
    PU.assert_errs(errs, "f64", "C1 full WENO9")


def test_weno79_argument_errors(binding, W):
    """halo < (order+1)/2, mixed orders and forcing the fused kernel are refused before anything is enqueued."""
    cfg = W.get_config("C1", size=(16, 16, 16), weno_order=9)
    gg = PU.gpu_grid(binding, cfg)
    st = gg.fields_from_state(W.generate_state(cfg))
    G = PU.new_G(binding, gg, cfg)
    p = dict(cfg["params"]); p["adv_x"] = 7
    with pytest.raises(binding.OcnError) as e:
        binding.ocn_compute_tendencies(gg, p, st, None, G)
    assert e.value.code == binding.OCN_ERR_UNSUPPORTED
    p = dict(cfg["params"]); p["adv_y"] = 5
    with pytest.raises(binding.OcnError) as e:
        binding.ocn_compute_tendencies(gg, p, st, None, G)
    assert e.value.code == binding.OCN_ERR_UNSUPPORTED
    cfg3 = W.get_config("C1", size=(16, 16, 16))                       # halo 3
    g3 = PU.gpu_grid(binding, cfg3)
    st3 = g3.fields_from_state(W.generate_state(cfg3))
    G3 = PU.new_G(binding, g3, cfg3)
    p = dict(cfg3["params"]); p["adv_x"] = p["adv_y"] = p["adv_z"] = 7
    with pytest.raises(binding.OcnError) as e:
        binding.ocn_compute_tendencies(g3, p, st3, None, G3)
    assert e.value.code == binding.OCN_ERR_INVALID
    gg.set_kernel(2)
    with pytest.raises(binding.OcnError) as e:
        binding.ocn_compute_tendencies(gg, cfg["params"], st, None, G)
    assert e.value.code == binding.OCN_ERR_UNSUPPORTED
