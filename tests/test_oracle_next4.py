"""Pins of the NEXT-4 oracle (six-dimensional sub-halo pass, Eq. 3; readings R29-R31).
CPU only.  Checked against things other than itself: scipy connected components of a numpy-built
float64 6-D adjacency (with a margin around the threshold), the sigma_v -> infinity limit (the
sub-halos of a halo found at linking length b are the halo itself), and a closed form (two
interpenetrating clumps with different bulk velocities separate in phase space only)."""
from __future__ import annotations

import numpy as np
from scipy.sparse import coo_matrix
from scipy.sparse.csgraph import connected_components

import oracle
from paper_2510_26851_b200 import inputs


def halos_with_velocities(seed=3):
    w = inputs.scaled(inputs.CONFIGS["cfg1"], 32)
    p = inputs.make_positions(w)
    rng = np.random.default_rng(seed)
    lab, _ = oracle.labels_cells(p, w.L, w.b)
    g = oracle.groups(p, lab, w.L, w.N_min)
    v = rng.standard_normal((len(p), 3)).astype(np.float32) * 50.0
    pg = g["particle_group"]
    half = (rng.random(len(p)) < 0.5) & (pg >= 0)     # half of every halo moves with a bulk flow
    v[half] += np.float32(400.0)
    return w, p, v, lab, g


def test_sigma_v_to_infinity_gives_back_the_halos():
    w, p, v, lab, g = halos_with_velocities()
    sub, E6 = oracle.subgroups(p, v, g["particle_group"], w.L, 1.0, 1e30, w.b)
    pg = g["particle_group"]
    assert np.array_equal(sub[pg >= 0], lab[pg >= 0])          # every kept halo is one sub-halo
    assert np.array_equal(sub[pg < 0], np.arange(len(p), dtype=np.int32)[pg < 0])   # R31
    assert E6 > 0


def _components(n, rows, cols):
    _, comp = connected_components(coo_matrix((np.ones(len(rows)), (rows, cols)), shape=(n, n)), directed=False)
    return comp


def _refines(fine, coarse):
    """every block of `fine` lies inside one block of `coarse`"""
    pairs = np.unique(np.stack([fine, coarse], 1), axis=0)
    return len(pairs) == len(np.unique(fine))


def test_against_scipy_components_of_a_float64_adjacency():
    """Float64 sandwich: the oracle's float32 partition is refined by the float64 components at
    ell (1 - delta) and refines those at ell (1 + delta); delta covers the float32 rounding of d2
    (a few 2^-24, plus L 2^-24 / |dx| for pairs that wrap)."""
    w, p, v, lab, g = halos_with_velocities(5)
    sx, sv, ell = 1.0, 120.0 ** 2, 1.3 * w.b
    sub, E6 = oracle.subgroups(p, v, g["particle_group"], w.L, sx, sv, ell)
    pg = g["particle_group"]
    n = len(p)
    x, vv = p.astype(np.float64), v.astype(np.float64)
    delta = 1e-5 + 8 * 2.0 ** -24 * (w.L / ell)
    edges = {-1: ([], []), 0: ([], []), 1: ([], [])}
    for k in range(g["K"]):
        mem = np.flatnonzero(pg == k)
        d = x[mem][:, None, :] - x[mem][None, :, :]
        d -= w.L * np.round(d / w.L)
        u = vv[mem][:, None, :] - vv[mem][None, :, :]
        d2 = np.triu((d ** 2).sum(-1) / sx + (u ** 2).sum(-1) / sv, 1) + np.tril(np.full((len(mem),) * 2, np.inf))
        for sgn in (-1, 0, 1):
            i, j = np.nonzero(d2 <= (ell * (1 + sgn * delta)) ** 2)
            edges[sgn][0].append(mem[i]); edges[sgn][1].append(mem[j])
    comps = {s: _components(n, np.concatenate(e[0]), np.concatenate(e[1])) for s, e in edges.items()}
    n_lo, n_hi = len(np.concatenate(edges[-1][0])), len(np.concatenate(edges[1][0]))
    assert n_lo <= E6 <= n_hi and n_hi - n_lo < 0.01 * E6
    assert _refines(comps[-1], sub) and _refines(sub, comps[1])
    assert sub.min() >= 0 and (sub <= np.arange(n)).all() and (sub[sub] == sub).all()   # canonical: min index
    assert len(np.unique(sub[pg >= 0])) > g["K"]               # the bulk flows do split halos


def test_two_streams_through_each_other_split_only_in_phase_space():
    rng = np.random.default_rng(8)
    L, b = 40.0, 1.0
    a = rng.standard_normal((60, 3)) * 0.3 + 20.0
    c = rng.standard_normal((60, 3)) * 0.3 + 20.0
    p = np.concatenate([a, c]).astype(np.float32)
    v = np.concatenate([np.full((60, 3), 100.0), np.full((60, 3), -100.0)]).astype(np.float32)
    v += rng.standard_normal(v.shape).astype(np.float32)
    lab, _ = oracle.labels_cells(p, L, b)
    assert (lab == 0).all()                                     # one halo in position space
    pg = np.zeros(len(p), np.int32)
    sub, _ = oracle.subgroups(p, v, pg, L, 1.0, 10.0 ** 2, b)  # velocity scale 10: the streams are 35 sigma apart
    assert (sub[:60] == 0).all() and (sub[60:] == 60).all()
    sub2, _ = oracle.subgroups(p, v, pg, L, 1.0, 1000.0 ** 2, b)   # velocity scale 1000: one sub-halo again
    assert (sub2 == 0).all()
