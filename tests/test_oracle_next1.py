"""Pins of the NEXT-1 oracle functions: halo decoration sigma (section 3.1.1,
reading R23) and the frozen-assignment backward (Eq. 4, Eq. 5).  CPU only.  Each pin
checks the oracle against something other than itself: numpy mean / std, closed forms, an exact
translation, and central finite differences of an independent numpy forward."""
from __future__ import annotations

import numpy as np
import pytest

import oracle
from paper_2510_26851_b200 import inputs


def clumps_away_from_faces(seed=5, L=64.0, b=1.0, sizes=(30, 45, 22, 60)):
    """Planted clumps (all members within b/2 of a centre, centres > 3 b apart, away from the faces);
    two more clumps of 5 and 7 members end up in dropped groups (N_min = 20)."""
    p, member = inputs.planted_cliques(seed, list(sizes) + [5, 7], L, b)
    assert (p > b).all() and (p < L - b).all()
    return np.ascontiguousarray(p, np.float32), member, L, b


def forward_numpy(p64, pg, K, mass):
    """Independent forward: plain (mass-weighted) mean and rms spread of each group, no wrap."""
    X = np.zeros((K, 3))
    S = np.zeros(K)
    for k in range(K):
        q, m = p64[pg == k], mass[pg == k]
        X[k] = (m[:, None] * q).sum(0) / m.sum()
        S[k] = np.sqrt((m * ((q - X[k]) ** 2).sum(1)).sum() / m.sum())
    return X, S


@pytest.mark.parametrize("weighted", [False, True])
def test_sigma_equals_numpy_std_away_from_faces(weighted):
    p, _, L, b = clumps_away_from_faces()
    lab, _ = oracle.labels_cells(p, L, b)
    m = np.random.default_rng(1).uniform(0.5, 1.5, len(p)).astype(np.float32) if weighted else None
    g = oracle.groups(p, lab, L, 20, mass=m)
    assert g["K"] == 4
    sig = oracle.group_sigma(p, g["particle_group"], L, g["group_com"], mass=m)
    X, S = forward_numpy(p.astype(np.float64), g["particle_group"], g["K"],
                         np.ones(len(p)) if m is None else m.astype(np.float64))
    assert np.allclose(g["group_com"], X, rtol=0, atol=1e-12 * L)
    assert np.allclose(sig, S, rtol=1e-12, atol=0)
    if m is None:   # unit masses: sigma^2 = sum of the three per-axis population variances
        for k in range(g["K"]):
            q = p[g["particle_group"] == k].astype(np.float64)
            assert np.isclose(sig[k] ** 2, q.var(0).sum(), rtol=1e-12)


def test_sigma_is_invariant_under_a_shift_across_the_face():
    """Exact float32 shift (positions on a 2^-10 lattice, L a power of two): the clump that now
    straddles the box face has the same sigma."""
    rng = np.random.default_rng(9)
    L, b = 64.0, 1.0
    q = (np.round((rng.standard_normal((40, 3)) * 0.2 + 32.0) * 1024) / 1024).astype(np.float32)
    shift = np.float32(31.75)                                     # centre moves to ~63.75: members wrap
    q2 = ((q + shift) % np.float32(L)).astype(np.float32)
    sig = []
    for pts in (q, q2):
        lab, _ = oracle.labels_cells(pts, L, b)
        g = oracle.groups(pts, lab, L, 20)
        assert g["K"] == 1 and g["group_size"][0] == 40
        sig.append(oracle.group_sigma(pts, g["particle_group"], L, g["group_com"])[0])
    assert (q2.max(0) - q2.min(0)).max() > L / 2                   # it really straddles a face
    assert abs(sig[0] - sig[1]) <= 1e-9


def test_backward_closed_forms():
    """Unit masses: dL/dx_i = G_g / N_g (Eq. 4).  Dropped particles get 0.  Weighted: m_i / M_g."""
    p, _, L, b = clumps_away_from_faces()
    lab, _ = oracle.labels_cells(p, L, b)
    g = oracle.groups(p, lab, L, 20)
    G = np.random.default_rng(2).standard_normal((g["K"], 3))
    d = oracle.groups_backward(p, g["particle_group"], L, g["group_mass"], g["group_com"], G)
    pg = g["particle_group"]
    assert (pg < 0).any() and (d[pg < 0] == 0).all()
    for k in range(g["K"]):
        assert np.allclose(d[pg == k], G[k] / g["group_size"][k], rtol=1e-15, atol=0)
        assert np.allclose(d[pg == k].sum(0), G[k], rtol=1e-12)       # the gradient is conserved
    m = np.random.default_rng(3).uniform(0.5, 1.5, len(p)).astype(np.float32)
    gw = oracle.groups(p, lab, L, 20, mass=m)
    dw = oracle.groups_backward(p, pg, L, gw["group_mass"], gw["group_com"], G, mass=m)
    for k in range(g["K"]):
        assert np.allclose(dw[pg == k], m[pg == k, None].astype(np.float64) / gw["group_mass"][k] * G[k], rtol=1e-14)


@pytest.mark.parametrize("weighted", [False, True])
def test_backward_matches_finite_differences_of_a_numpy_forward(weighted):
    """L(x) = sum_g a_g . X_g(x) + c_g sigma_g(x) at frozen membership; central differences in float64
    of the numpy forward against the oracle's analytic backward (through X and through sigma)."""
    p, _, L, b = clumps_away_from_faces(seed=11, sizes=(25, 33))
    lab, _ = oracle.labels_cells(p, L, b)
    rng = np.random.default_rng(4)
    m32 = rng.uniform(0.5, 1.5, len(p)).astype(np.float32) if weighted else None
    m64 = np.ones(len(p)) if m32 is None else m32.astype(np.float64)
    g = oracle.groups(p, lab, L, 20, mass=m32)
    K, pg = g["K"], g["particle_group"]
    sig = oracle.group_sigma(p, pg, L, g["group_com"], mass=m32)
    a, c = rng.standard_normal((K, 3)), rng.standard_normal(K)
    grad = oracle.groups_backward(p, pg, L, g["group_mass"], g["group_com"], a, group_sigma=sig, grad_sigma=c,
                                  mass=m32)

    def loss(x):
        X, S = forward_numpy(x, pg, K, m64)
        return (a * X).sum() + (c * S).sum()

    x0 = p.astype(np.float64)
    eps = 1e-6
    members = np.flatnonzero(pg >= 0)
    for i in rng.choice(members, size=12, replace=False):
        for ax in range(3):
            xp, xm = x0.copy(), x0.copy()
            xp[i, ax] += eps
            xm[i, ax] -= eps
            fd = (loss(xp) - loss(xm)) / (2 * eps)
            assert abs(fd - grad[i, ax]) <= 1e-7 * max(1.0, abs(fd)), (i, ax, fd, grad[i, ax])
    # only through sigma: the gradient of a group sums to zero (sigma is translation invariant)
    gs = oracle.groups_backward(p, pg, L, g["group_mass"], g["group_com"], np.zeros((K, 3)), group_sigma=sig,
                                grad_sigma=c, mass=m32)
    for k in range(K):
        assert np.abs(gs[pg == k].sum(0)).max() <= 1e-12
