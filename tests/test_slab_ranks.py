"""Multi-GPU y-slabs (include/ocn.h ocn_grid_set_external_halo), the host side on CPU: world_size-2 and -3 `gloo`
process groups exchange the H outermost rows of dense padded fields through `paper_2502_14148_b200.slab.YSlabs` — the same
partition, neighbour and transport code the GPU path uses (there the packing is done by libocn's kernels) — and every rank's
padded slab must equal the corresponding rows (periodic wrap, corners included) of the global field; then the ORACLE advances
each slab by a full substage and the interiors must equal the oracle's global result bit for bit (the path shards with no
data-path collective beyond that neighbour exchange)."""
import os
import socket
import sys

import numpy as np
import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
H = 3
NX, NY, NZ = 9, 14, 5


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _global_fields(nf=3):
    rng = np.random.default_rng(4242)
    return [rng.standard_normal((NZ, NY, NX)) for _ in range(nf)]


def _pad_xz(a):
    """periodic x, mirrored (no-flux) z halos of an (nz, ny, nx) block; y is left without halo"""
    a = np.concatenate([a[:, :, -H:], a, a[:, :, :H]], axis=2)
    lo = a[:H][::-1]
    hi = a[-H:][::-1]
    return np.concatenate([lo, a, hi], axis=0)


def _worker(rank, world, port, ny, out):
    import torch
    import torch.distributed as dist
    sys.path.insert(0, ROOT)
    from paper_2502_14148_b200.slab import YSlabs
    dist.init_process_group("gloo", init_method="tcp://127.0.0.1:%d" % port, rank=rank, world_size=world)
    sl = YSlabs(ny, H, world, rank)
    glob = [g[:, :ny, :] for g in _global_fields()]
    fields = []
    for g in glob:
        loc = _pad_xz(g[:, sl.local_slice(), :])
        full = np.full((loc.shape[0], sl.ny_local + 2 * H, loc.shape[2]), np.nan)
        full[:, H:H + sl.ny_local, :] = loc
        fields.append(torch.from_numpy(full))
    sl.exchange_dense(fields)
    ok = True
    rows = sl.global_rows()
    for f, g in zip(fields, glob):
        want = _pad_xz(g)[:, rows, :]
        ok = ok and np.array_equal(f.numpy(), want)
    out.put((rank, ok, sl.j0, sl.ny_local, sl.south, sl.north))
    dist.barrier()
    dist.destroy_process_group()


@pytest.mark.parametrize("world,ny", [(2, 14), (2, 13), (3, 14)])
def test_slab_exchange_gloo(world, ny):
    import torch.multiprocessing as mp
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = _free_port()
    procs = [ctx.Process(target=_worker, args=(r, world, port, ny, q)) for r in range(world)]
    for p in procs:
        p.start()
    res = sorted(q.get(timeout=180) for _ in procs)
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    assert [r[1] for r in res] == [True] * world, res
    assert sum(r[3] for r in res) == ny and [r[2] for r in res] == [sum(x[3] for x in res[:k]) for k in range(world)]
    for rank, _, _, _, south, north in res:
        assert south == (rank - 1) % world and north == (rank + 1) % world


def test_partition_rules():
    sys.path.insert(0, ROOT)
    from paper_2502_14148_b200.slab import YSlabs
    s = YSlabs(512, 3, 8, 5)
    assert (s.j0, s.ny_local, s.south, s.north) == (320, 64, 4, 6)
    s = YSlabs(10, 3, 3, 0)                      # uneven: 4, 3, 3
    assert s.counts == [4, 3, 3] and s.global_rows() == [7, 8, 9, 0, 1, 2, 3, 4, 5, 6]
    with pytest.raises(ValueError):
        YSlabs(8, 3, 3, 0)                       # a slab would be thinner than the halo
    with pytest.raises(NotImplementedError):
        YSlabs(64, 3, 2, 0, periodic=False)      # walls on a slab boundary: not built
    one = YSlabs(12, 3, 1, 0)                    # a single slab is its own periodic neighbour
    import torch
    f = torch.arange(2 * 18 * 4, dtype=torch.float64).reshape(2, 18, 4).clone()
    g = f.clone()
    one.exchange_dense([f])
    assert torch.equal(f[:, :3], g[:, 12:15]) and torch.equal(f[:, 15:], g[:, 3:6])


def test_slabs_advance_like_the_global_grid_with_the_oracle(ref):
    """two slabs, each advanced by the ORACLE with y halos taken from the neighbour (Periodic local topology on a padded
    array whose y halos were overwritten by the exchange rule), reproduce the oracle's global substage bit for bit."""
    sys.path.insert(0, ROOT)
    from paper_2502_14148_b200.slab import YSlabs
    from paper_2502_14148_b200 import workloads as W
    cfg = W.get_config("C1", size=(12, 16, 6))
    p, g = cfg["params"], cfg["grid"]
    state = W.generate_state(cfg)
    rg = ref.RefGrid(g["Nx"], g["Ny"], g["Nz"], H, g["dx"], g["dy"], g["dz_c"], g["dz_uniform"], g["topology"])
    glob = {"u": state["u"].copy(), "v": state["v"].copy(), "w": state["w"].copy(), "c": [c.copy() for c in state["c"]]}
    ref.fill_halos(rg, p, glob)
    Gg = ref.compute_tendencies(rg, p, glob)
    for rank in range(2):
        sl = YSlabs(g["Ny"], H, 2, rank)
        rows = sl.global_rows()
        lg = ref.RefGrid(g["Nx"], sl.ny_local, g["Nz"], H, g["dx"], g["dy"], g["dz_c"], g["dz_uniform"], g["topology"])
        take = lambda a: np.ascontiguousarray(a[:, [r + H for r in rows], :])      # global padded rows -> slab rows (wrap)
        loc = {"u": take(glob["u"]), "v": take(glob["v"]), "w": take(glob["w"]), "c": [take(c) for c in glob["c"]]}
        Gl = ref.compute_tendencies(lg, p, loc)
        for k in ("u", "v", "w"):
            assert np.array_equal(lg.interior(Gl[k]), rg.interior(Gg[k])[:, sl.local_slice(), :]), (rank, k)
        for a, b in zip(Gl["c"], Gg["c"]):
            assert np.array_equal(lg.interior(a), rg.interior(b)[:, sl.local_slice(), :])
