"""y-slab decomposition of the hot path over several GPUs (App. C "slab and pencil decomposition").

One process per GPU (torch.distributed; NCCL between GPUs, gloo in the CPU tests) owns a contiguous slab of rows of a grid
that is Periodic in y.  The path shards naturally — tendencies are local stencils of reach H, the substage is pointwise, the
column scans are local to a column — so the ONLY exchange is one neighbour step per halo fill: every rank sends the H
outermost interior rows of each side of every prognostic field to the neighbour on that side (C2 split in y: 3 x 528 x 262
x 8 B = 3.3 MB per field per direction) and receives its own halo rows.  No reduction, no all-to-all.

Argument marshalling and transport only: the packing / unpacking of device buffers is done by libocn's kernels
(ocn_halo_pack_y / ocn_halo_unpack_y); the CPU methods on dense arrays (`exchange_dense`) are the same index arithmetic written
with slices and exist so that the partition / neighbour logic can be tested with world_size-2 gloo runs without a GPU.
"""
import torch
import torch.distributed as dist


class YSlabs:
    def __init__(self, Ny_global, halo, world=1, rank=0, periodic=True):
        if not periodic:
            raise NotImplementedError("y-slabs with walls on a slab boundary are not built (include/ocn.h ocn_grid_set_external_halo)")
        if world < 1 or not (0 <= rank < world):
            raise ValueError("bad world/rank")
        self.Ny, self.H, self.world, self.rank = int(Ny_global), int(halo), int(world), int(rank)
        base, extra = divmod(self.Ny, self.world)
        counts = [base + (1 if r < extra else 0) for r in range(self.world)]
        if min(counts) < self.H:
            raise ValueError("every slab needs at least halo=%d rows (Ny=%d over %d ranks)" % (self.H, self.Ny, self.world))
        self.counts = counts
        self.j0 = sum(counts[:rank])                 # 0-based global index of the first local row
        self.ny_local = counts[rank]
        self.south = (rank - 1) % world              # neighbour holding rows below j0 (Periodic wrap)
        self.north = (rank + 1) % world

    # ------------------------------------------------------------------ which global rows a slab sees
    def global_rows(self, with_halo=True):
        """global (wrapped) row index of every local row, halos included: what the slab's padded array must equal."""
        lo = self.j0 - (self.H if with_halo else 0)
        hi = self.j0 + self.ny_local + (self.H if with_halo else 0)
        return [j % self.Ny for j in range(lo, hi)]

    def local_slice(self):
        return slice(self.j0, self.j0 + self.ny_local)

    def local_params(self, params, dy):
        """the parameter dict THIS slab's kernels must be given: libocn evaluates the beta-plane Coriolis parameter
        f = f0 + beta (y_j - y0) from the local row index, so the slab's y-origin moves down by the j0 rows below it
        (include/ocn.h, ocn_grid_set_external_halo).  Everything else is shared by all ranks."""
        return dict(params, y0=float(params.get("y0", 0.0)) - self.j0 * float(dy))

    # ------------------------------------------------------------------ transport
    def _swap(self, send_lo, send_hi, recv_lo, recv_hi, group=None):
        """send_lo -> south neighbour's high halo, send_hi -> north neighbour's low halo; receive ours.  world == 1: the slab is its
        own periodic neighbour (plain copies)."""
        if self.world == 1:
            recv_lo.copy_(send_hi)
            recv_hi.copy_(send_lo)
            return
        if self.world == 2:
            # both neighbours are the SAME peer.  NCCL ignores P2P tags and pairs the messages between two ranks purely by issue
            # order, so nothing here may depend on tags: one message per direction, [low rows | high rows] in one buffer.
            peer = self.north
            out = torch.cat([send_lo.reshape(-1), send_hi.reshape(-1)])
            inn = torch.empty_like(out)
            for r in dist.batch_isend_irecv([dist.P2POp(dist.isend, out, peer, group=group), dist.P2POp(dist.irecv, inn, peer, group=group)]):
                r.wait()
            n = send_lo.numel()
            recv_hi.reshape(-1).copy_(inn[:n])       # the peer's low rows are our high halo
            recv_lo.reshape(-1).copy_(inn[n:])       # the peer's high rows are our low halo
            return
        # world >= 3: south and north are different peers, exactly one message per (peer, direction) — no pairing ambiguity, no tags
        ops = [dist.P2POp(dist.isend, send_lo, self.south, group=group),
               dist.P2POp(dist.isend, send_hi, self.north, group=group),
               dist.P2POp(dist.irecv, recv_hi, self.north, group=group),     # the north neighbour's low rows
               dist.P2POp(dist.irecv, recv_lo, self.south, group=group)]     # the south neighbour's high rows
        for r in dist.batch_isend_irecv(ops):
            r.wait()

    # ------------------------------------------------------------------ device path: libocn kernels + torch.distributed
    def make_buffers(self, B, grid, params):
        n = B.ocn_halo_slab_elems(grid, params)
        mk = lambda: torch.empty(n, dtype=grid.tdtype, device=grid.device)
        return {"send_lo": mk(), "send_hi": mk(), "recv_lo": mk(), "recv_hi": mk()}

    def exchange(self, B, grid, params, state, bufs, group=None):
        """after ocn_fill_halos (x and z halos; the grid is marked ocn_grid_set_external_halo(1)): fill the y halos of `state`."""
        B.ocn_halo_pack_y(grid, params, state, 0, bufs["send_lo"])
        B.ocn_halo_pack_y(grid, params, state, 1, bufs["send_hi"])
        self._swap(bufs["send_lo"], bufs["send_hi"], bufs["recv_lo"], bufs["recv_hi"], group)
        B.ocn_halo_unpack_y(grid, params, state, 0, bufs["recv_lo"])
        B.ocn_halo_unpack_y(grid, params, state, 1, bufs["recv_hi"])

    # ------------------------------------------------------------------ dense CPU path (tests of the host logic)
    def exchange_dense(self, fields, group=None):
        """fields: list of dense padded CPU tensors (nz_pad, ny_local + 2H, nx_pad), x / z halos already filled."""
        H, n = self.H, self.ny_local
        send_lo = torch.stack([f[:, H:2 * H, :] for f in fields]).contiguous()
        send_hi = torch.stack([f[:, n:n + H, :] for f in fields]).contiguous()
        recv_lo, recv_hi = torch.empty_like(send_lo), torch.empty_like(send_hi)
        self._swap(send_lo, send_hi, recv_lo, recv_hi, group)
        for t, f in enumerate(fields):
            f[:, 0:H, :] = recv_lo[t]
            f[:, n + H:n + 2 * H, :] = recv_hi[t]
