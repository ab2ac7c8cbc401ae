"""Slab-decomposed multi-GPU Friends-of-Friends (section 2.3).

The box is cut into `world` slabs along z; rank r owns z in [r L / world, (r + 1) L / world).  Every
rank borrows the lower boundary layer (a little more than b thick) of the rank above it (periodic
ring), links own + ghost particles with the single-GPU path, turns its local labels into
minimum-GLOBAL-id labels, learns what the owner of each ghost calls that ghost's group, and the
resulting label equivalences — all-gathered, a few thousand pairs — are merged by one union-find that
every rank runs on its own copy.  The result for the particles a rank owns is identical to a
monolithic run on the whole box ("minimum global particle ID").

Only labels are produced (group reductions across ranks are not built).  Every step that touches
particles or pairs runs in kernels of libfof_b200.so (fof_layer_select, fof_link, fof_component_min,
fof_merge_labels); this module only moves tensors between ranks with torch.distributed (two ring
send/recv rounds and one all-gather) — plumbing.  The phases are separate methods so that a single
process can play all ranks in turn (tests on one GPU); `slab_fof` is the one-process-per-GPU driver.
"""
from __future__ import annotations

import numpy as np

from . import binding as B

GHOST_MARGIN = 1.001  # ghost layer = b * GHOST_MARGIN thick: covers the float32 rounding of the face distance


class SlabRank:
    """One rank's share of the work, in four local phases separated by three exchanges."""

    def __init__(self, pos, ids, L: float, b: float, rank: int, world: int, n_global: int):
        import torch

        assert world >= 2, "one slab is the monolithic path: call FoF.link"
        assert L / world >= 3.0 * b * GHOST_MARGIN, "slabs must be at least three ghost layers thick"
        assert pos.is_cuda and pos.dtype == torch.float32 and pos.dim() == 2 and pos.shape[1] == 3
        assert ids.dtype == torch.int32 and ids.shape[0] == pos.shape[0]
        self.pos, self.ids = pos.contiguous(), ids.contiguous()
        self.L, self.b, self.rank, self.world, self.n_global = float(L), float(b), rank, world, int(n_global)
        self.dev = pos.device
        self.n_own = pos.shape[0]

    # ---- phase A: my lower boundary layer, to be lent to the rank below ---------------------------------
    def ghosts_to_send(self):
        import torch

        idx = torch.empty(max(self.n_own, 1), dtype=torch.int32, device=self.dev)
        cnt = torch.zeros(1, dtype=torch.int32, device=self.dev)
        z_lo = np.float32(self.rank * (self.L / self.world))
        B.fof_layer_select(self.pos, self.L, 2, float(z_lo), float(np.float32(self.b * GHOST_MARGIN)), idx, cnt)
        self.sent_idx = idx[: int(cnt.item())].long()
        return self.pos[self.sent_idx].contiguous(), self.ids[self.sent_idx].contiguous()

    # ---- phase B: link own + borrowed particles; labels in global ids -------------------------------------
    def link(self, ghost_pos, ghost_ids):
        import torch

        self.n_ghost = ghost_pos.shape[0]
        pos = torch.cat([self.pos, ghost_pos.to(self.dev)]).contiguous()
        ids = torch.cat([self.ids, ghost_ids.to(self.dev)]).contiguous()
        n = pos.shape[0]
        f = B.FoF(n, self.L, self.b, 1, device=self.dev)
        local = f.link(pos)
        f.close()
        tmp = torch.empty(max(n, 1), dtype=torch.int32, device=self.dev)
        self.glabel = torch.empty(max(n, 1), dtype=torch.int32, device=self.dev)[:n]
        B.fof_component_min(local, ids, tmp, self.glabel)
        # what I call the groups of the particles I lent out (same order as ghosts_to_send)
        return self.glabel[self.sent_idx].contiguous()

    # ---- phase C: equivalences between my labels and the owner's labels of the borrowed particles ----
    def equivalences(self, owner_labels):
        import torch

        mine = self.glabel[self.n_own:self.n_own + self.n_ghost]
        theirs = owner_labels.to(self.dev)
        keep = mine != theirs
        return torch.stack([mine[keep], theirs[keep]], 1).contiguous()

    # ---- phase D: merge all equivalences, relabel the particles I own ---------------------------------------
    def merge(self, all_pairs):
        import torch

        labels = self.glabel[: self.n_own].clone()
        parent = torch.empty(max(self.n_global, 1), dtype=torch.int32, device=self.dev)[: self.n_global]
        B.fof_merge_labels(all_pairs.to(self.dev).contiguous(), parent, labels)
        return labels


# ------------------------------------------------------------------------------------------------ exchange
class RingExchange:
    """Variable-length ring send/recv and all-gather over torch.distributed (nccl or gloo)."""

    def __init__(self, group=None):
        import torch.distributed as dist

        self.dist, self.group = dist, group
        self.rank, self.world = dist.get_rank(group), dist.get_world_size(group)

    def send_down_recv_up(self, t):
        """Send rows of `t` to rank - 1, return the rows rank + 1 sent (periodic ring)."""
        import torch

        dist = self.dist
        down, up = (self.rank - 1) % self.world, (self.rank + 1) % self.world
        n_out = torch.tensor([t.shape[0]], dtype=torch.int64, device=t.device)
        n_in = torch.zeros(1, dtype=torch.int64, device=t.device)
        reqs = [dist.isend(n_out, down, group=self.group), dist.irecv(n_in, up, group=self.group)]
        for r in reqs:
            r.wait()
        buf = torch.empty((int(n_in.item()),) + tuple(t.shape[1:]), dtype=t.dtype, device=t.device)
        reqs = []
        if t.shape[0]:
            reqs.append(dist.isend(t.contiguous(), down, group=self.group))
        if buf.shape[0]:
            reqs.append(dist.irecv(buf, up, group=self.group))
        for r in reqs:
            r.wait()
        return buf

    def all_gather_rows(self, t):
        import torch

        dist = self.dist
        n = torch.tensor([t.shape[0]], dtype=torch.int64, device=t.device)
        sizes = [torch.zeros_like(n) for _ in range(self.world)]
        dist.all_gather(sizes, n, group=self.group)
        sizes = [int(s.item()) for s in sizes]
        m = max(max(sizes), 1)
        pad = torch.zeros((m,) + tuple(t.shape[1:]), dtype=t.dtype, device=t.device)
        pad[: t.shape[0]] = t
        bufs = [torch.empty_like(pad) for _ in range(self.world)]
        dist.all_gather(bufs, pad, group=self.group)
        return torch.cat([b[:s] for b, s in zip(bufs, sizes)])


def slab_fof(pos, ids, L: float, b: float, n_global: int, group=None):
    """One process per GPU: `pos` / `ids` are the particles this rank owns (its z slab) and their global
    ids; returns their labels = minimum global id of the group, identical to a monolithic run."""
    ex = RingExchange(group)
    me = SlabRank(pos, ids, L, b, ex.rank, ex.world, n_global)
    gpos, gids = me.ghosts_to_send()
    rpos, rids = ex.send_down_recv_up(gpos), ex.send_down_recv_up(gids)
    lent_labels = me.link(rpos, rids)
    owner_labels = ex.send_down_recv_up(lent_labels)
    pairs = ex.all_gather_rows(me.equivalences(owner_labels))
    return me.merge(pairs)


def slab_fof_emulated(parts, L: float, b: float, n_global: int):
    """All ranks played in turn by one process on one device (tests): parts = [(pos, ids)] per slab."""
    import torch

    world = len(parts)
    ranks = [SlabRank(p, i, L, b, r, world, n_global) for r, (p, i) in enumerate(parts)]
    sent = [rk.ghosts_to_send() for rk in ranks]
    lent = [rk.link(*sent[(r + 1) % world]) for r, rk in enumerate(ranks)]
    pairs = torch.cat([rk.equivalences(lent[(r + 1) % world]) for r, rk in enumerate(ranks)])
    return [rk.merge(pairs) for rk in ranks]


def slab_faces(L: float, world: int):
    """Lower faces of the slabs as float32, the same expression SlabRank.ghosts_to_send uses: ownership
    and ghost selection must agree bit for bit on which side of a face a particle lies."""
    return np.array([np.float32(r * (L / world)) for r in range(world)], dtype=np.float32)


def split_into_slabs(pos_np, L: float, world: int):
    """Host helper for tests / examples: indices of the particles of each z slab.  Positions must already
    lie in [0, L) (float32); rank r owns faces[r] <= z < faces[r + 1]."""
    z = np.asarray(pos_np[:, 2], dtype=np.float32)
    assert (z >= 0).all() and (z < np.float32(L)).all()
    owner = np.searchsorted(slab_faces(L, world), z, side="right") - 1
    return [np.flatnonzero(owner == r) for r in range(world)]
