"""Slab-decomposed multi-GPU Friends-of-Friends (section 2.3).

The box is cut into `world` slabs along z; rank r owns z in [r L / world, (r + 1) L / world).  Every
rank borrows the lower boundary layer (a little more than b thick) of the rank above it (periodic
ring), links own + ghost particles with the single-GPU path, turns its local labels into
minimum-GLOBAL-id labels, learns what the owner of each ghost calls that ghost's group, and the
resulting label equivalences — all-gathered, a few thousand pairs — are merged by one union-find that
every rank runs on its own copy.  The result for the particles a rank owns is identical to a
monolithic run on the whole box ("minimum global particle ID").

Groups (sizes, masses, periodic centres of mass) follow the same way: a group that spans ranks shows up
among the final labels of the borrowed particles; the owners of the canonical particles of those groups
publish their positions, every rank runs the single-GPU fof_groups on its own particles plus one massless
proxy per foreign canonical particle (so its members are unwrapped relative to the same reference as in a
monolithic run), and the partial records of the spanning groups are gathered and combined by the owner of
the canonical particle (fof_combine_groups).  The catalogue of a rank = the groups whose canonical particle
it owns; the union over ranks, ordered by label, is the monolithic catalogue.

Every step that touches particles, pairs or group records runs in kernels of libfof_b200.so
(fof_layer_select, fof_link, fof_component_min, fof_merge_labels_sparse, fof_groups, fof_combine_groups);
this module moves tensors between ranks with torch.distributed (two ring send/recv rounds and four
all-gathers of a few thousand rows) and builds index lists with torch sort / unique / searchsorted —
plumbing.  The phases are separate methods so that a single process can play all ranks in turn (tests on
one GPU); `slab_fof` / `slab_fof_groups` are the one-process-per-GPU drivers.
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

    # ---- phase D: merge all equivalences, relabel the particles I own (and the ones I borrowed) -----------------
    def merge(self, all_pairs):
        """Union-find over the DISTINCT labels that occur in the pairs (a few thousand), not over all global ids."""
        import torch

        n = self.n_own + self.n_ghost
        final = self.glabel[:n].clone()
        pairs = all_pairs.to(self.dev).contiguous()
        if pairs.shape[0]:
            uniq = torch.unique(pairs.reshape(-1))  # ascending
            parent = torch.empty(uniq.shape[0], dtype=torch.int32, device=self.dev)
            B.fof_merge_labels_sparse(pairs, uniq.contiguous(), parent, final)
        self.labels = final[: self.n_own]
        self.ghost_labels = final[self.n_own:]
        return self.labels

    # ---- groups, phase E: labels of the groups that may span ranks (every such group holds a borrowed particle) --
    def ghost_group_labels(self):
        import torch

        return torch.unique(self.ghost_labels)

    # ---- phase F: positions of the canonical particles I own among those groups -------------------------------------
    def refs_for(self, spanning):
        import torch

        sid, perm = torch.sort(self.ids)
        p = torch.searchsorted(sid, spanning).clamp_(max=max(self.n_own - 1, 0))
        mine = (sid[p] == spanning) if self.n_own else torch.zeros_like(spanning, dtype=torch.bool)
        self._sid, self._perm = sid, perm
        return spanning[mine].contiguous(), self.pos[perm[p[mine]]].contiguous()

    # ---- phase G: fof_groups on my own particles + one massless proxy per foreign canonical particle ----------------
    def local_groups(self, spanning, ref_labels, ref_pos, mass=None, N_min: int = 1):
        """Returns the partial records of the spanning groups I hold members of, one row per group:
        float64 [k, 6] = (label, members, mass, cx, cy, cz)."""
        import torch

        dev, n_own = self.dev, self.n_own
        uniq, inv = torch.unique(self.labels, return_inverse=True)
        sid, perm = self._sid, self._perm
        p = torch.searchsorted(sid, uniq).clamp_(max=max(n_own - 1, 0))
        own = (sid[p] == uniq) if n_own else torch.zeros_like(uniq, dtype=torch.bool)
        foreign = uniq[~own]
        order = torch.argsort(ref_labels)
        rl, rp = ref_labels[order], ref_pos[order]
        q = torch.searchsorted(rl, foreign).clamp_(max=max(rl.shape[0] - 1, 0))
        assert foreign.shape[0] == 0 or bool((rl[q] == foreign).all()), "a foreign canonical particle without a published position"
        canon = torch.empty(uniq.shape[0], dtype=torch.int64, device=dev)
        canon[own] = perm[p[own]]
        canon[~own] = n_own + torch.arange(foreign.shape[0], device=dev)
        n_aug = n_own + foreign.shape[0]
        pos = torch.cat([self.pos, rp[q]]).contiguous()
        m_own = mass.to(dev) if mass is not None else torch.ones(n_own, dtype=torch.float32, device=dev)
        m_aug = torch.cat([m_own, torch.zeros(foreign.shape[0], dtype=torch.float32, device=dev)]).contiguous()
        lab_local = torch.cat([canon[inv], n_own + torch.arange(foreign.shape[0], device=dev)]).to(torch.int32).contiguous()
        ids_aug = torch.cat([self.ids, foreign.to(torch.int32)])
        self.N_min, self.has_mass = int(N_min), mass is not None
        if n_aug == 0:
            self._loc = None
            return torch.zeros((0, 6), dtype=torch.float64, device=dev)
        f = B.FoF(n_aug, self.L, self.b, 1, device=dev)
        g = f.groups(pos, lab_local, mass=m_aug)
        f.close()
        glab = ids_aug[g["group_label"].long()]                                  # global label of every local group
        size = g["group_size"] - (g["group_label"] >= n_own).to(torch.int32)    # the proxy is not a member
        sp = torch.searchsorted(spanning, glab).clamp_(max=max(spanning.shape[0] - 1, 0))
        is_span = (spanning[sp] == glab) if spanning.shape[0] else torch.zeros_like(glab, dtype=torch.bool)
        self._loc = dict(label=glab, size=size, mass=g["group_mass"], com=g["group_com"], span=is_span,
                         owned=g["group_label"] < n_own, canon_pos=pos[g["group_label"].long()])
        rows = torch.cat([glab[is_span, None].double(), size[is_span, None].double(), g["group_mass"][is_span, None].double(),
                          g["group_com"][is_span].double()], 1)
        return rows.contiguous()

    # ---- phase H: the catalogue of the groups whose canonical particle I own -----------------------------------------
    def finish_groups(self, all_rows):
        import torch

        dev = self.dev
        loc = self._loc
        if loc is None:
            z = torch.zeros(0, device=dev)
            return dict(K=0, group_label=z.int(), group_size=z.int(), group_mass=z.float(), group_com=torch.zeros((0, 3), device=dev))
        rows = all_rows.to(dev)
        rows = rows[torch.argsort(rows[:, 0])]
        part_label = rows[:, 0].to(torch.int32).contiguous()
        part_size = rows[:, 1].to(torch.int32).contiguous()
        part_mass = rows[:, 2].to(torch.float32).contiguous()
        part_com = rows[:, 3:6].to(torch.float32).contiguous()
        mine = loc["span"] & loc["owned"]
        want = loc["label"][mine].to(torch.int32).contiguous()
        W = want.shape[0]
        o_size = torch.empty(W, dtype=torch.int32, device=dev)
        o_mass = torch.empty(W, dtype=torch.float32, device=dev)
        o_com = torch.empty((W, 3), dtype=torch.float32, device=dev)
        if W:
            B.fof_combine_groups(want, loc["canon_pos"][mine].contiguous(), self.L, part_label, part_size, part_mass,
                                 part_com, o_size, o_mass, o_com)
        solo = ~loc["span"]   # groups no other rank holds a member of: fof_groups' record is final
        label = torch.cat([loc["label"][solo].to(torch.int32), want])
        size = torch.cat([loc["size"][solo], o_size])
        gmass = torch.cat([loc["mass"][solo], o_mass])
        com = torch.cat([loc["com"][solo], o_com])
        keep = size >= self.N_min
        order = torch.argsort(label[keep])
        return dict(K=int(keep.sum().item()), group_label=label[keep][order], group_size=size[keep][order],
                    group_mass=gmass[keep][order], group_com=com[keep][order])


# ------------------------------------------------------------------------------------------------ exchange
class RingExchange:
    """Variable-length ring send/recv and all-gather over torch.distributed (nccl or gloo)."""

    def __init__(self, group=None):
        import torch.distributed as dist

        self.dist, self.group = dist, group
        self.rank, self.world = dist.get_rank(group), dist.get_world_size(group)
        self.stage_on_host = dist.get_backend(group) == "gloo"  # gloo moves host tensors only (CPU tests, one-GPU checks)

    def send_down_recv_up(self, t):
        """Send rows of `t` to rank - 1, return the rows rank + 1 sent (periodic ring)."""
        import torch

        dist = self.dist
        home = t.device
        if self.stage_on_host:
            t = t.cpu()
        down, up = (self.rank - 1) % self.world, (self.rank + 1) % self.world
        n_out = torch.tensor([t.shape[0]], dtype=torch.int64, device=t.device)
        n_in = torch.zeros(1, dtype=torch.int64, device=t.device)
        # send and receive posted as ONE batch: with nccl a lone isend may wait for the peer's recv, which is queued
        # behind the peer's own send (every rank sends first) -- only grouped pairs are guaranteed to progress
        ops = [dist.P2POp(dist.isend, n_out, down, self.group), dist.P2POp(dist.irecv, n_in, up, self.group)]
        for r in dist.batch_isend_irecv(ops):
            r.wait()
        buf = torch.empty((int(n_in.item()),) + tuple(t.shape[1:]), dtype=t.dtype, device=t.device)
        ops = []
        if t.shape[0]:
            ops.append(dist.P2POp(dist.isend, t.contiguous(), down, self.group))
        if buf.shape[0]:
            ops.append(dist.P2POp(dist.irecv, buf, up, self.group))
        if ops:
            for r in dist.batch_isend_irecv(ops):
                r.wait()
        return buf.to(home)

    def all_gather_rows(self, t):
        import torch

        dist = self.dist
        home = t.device
        if self.stage_on_host:
            t = t.cpu()
        n = torch.tensor([t.shape[0]], dtype=torch.int64, device=t.device)
        sizes = [torch.zeros_like(n) for _ in range(self.world)]
        dist.all_gather(sizes, n, group=self.group)
        sizes = [int(s.item()) for s in sizes]
        m = max(max(sizes), 1)
        pad = torch.zeros((m,) + tuple(t.shape[1:]), dtype=t.dtype, device=t.device)
        pad[: t.shape[0]] = t
        bufs = [torch.empty_like(pad) for _ in range(self.world)]
        dist.all_gather(bufs, pad, group=self.group)
        return torch.cat([b[:s] for b, s in zip(bufs, sizes)]).to(home)


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


def slab_fof_groups(pos, ids, L: float, b: float, n_global: int, N_min: int = 20, mass=None, group=None):
    """One process per GPU: labels of the particles this rank owns plus the catalogue (label, size, mass, periodic
    centre of mass) of the groups whose canonical particle it owns.  Returns (labels, groups dict)."""
    import torch

    ex = RingExchange(group)
    me = SlabRank(pos, ids, L, b, ex.rank, ex.world, n_global)
    gpos, gids = me.ghosts_to_send()
    rpos, rids = ex.send_down_recv_up(gpos), ex.send_down_recv_up(gids)
    lent_labels = me.link(rpos, rids)
    owner_labels = ex.send_down_recv_up(lent_labels)
    labels = me.merge(ex.all_gather_rows(me.equivalences(owner_labels)))
    spanning = torch.unique(ex.all_gather_rows(me.ghost_group_labels()))
    rl, rp = me.refs_for(spanning)
    rows = me.local_groups(spanning, ex.all_gather_rows(rl), ex.all_gather_rows(rp), mass=mass, N_min=N_min)
    return labels, me.finish_groups(ex.all_gather_rows(rows))


def slab_fof_emulated(parts, L: float, b: float, n_global: int, N_min=None, masses=None):
    """All ranks played in turn by one process on one device (tests): parts = [(pos, ids)] per slab.  Returns the
    labels per slab, and with N_min given also the catalogue per slab (masses: per-slab tensors or None)."""
    import torch

    world = len(parts)
    ranks = [SlabRank(p, i, L, b, r, world, n_global) for r, (p, i) in enumerate(parts)]
    sent = [rk.ghosts_to_send() for rk in ranks]
    lent = [rk.link(*sent[(r + 1) % world]) for r, rk in enumerate(ranks)]
    pairs = torch.cat([rk.equivalences(lent[(r + 1) % world]) for r, rk in enumerate(ranks)])
    labels = [rk.merge(pairs) for rk in ranks]
    if N_min is None:
        return labels
    spanning = torch.unique(torch.cat([rk.ghost_group_labels() for rk in ranks]))
    refs = [rk.refs_for(spanning) for rk in ranks]
    rl, rp = torch.cat([r[0] for r in refs]), torch.cat([r[1] for r in refs])
    rows = torch.cat([rk.local_groups(spanning, rl, rp, mass=None if masses is None else masses[r], N_min=N_min)
                      for r, rk in enumerate(ranks)])
    return labels, [rk.finish_groups(rows) for rk in ranks]


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
