"""Pins of the NEXT-3 oracle (stochastic-edge FoF, section 3.2 Eq. 6-8; readings R25-R28 of
DESIGN.md).  CPU only.  The oracle is checked against things other than itself: numpy's logistic,
the deterministic FoF oracle in the alpha -> infinity limit, scipy connected components of the listed
edges, binomial statistics of the sampled edges, the textbook Bernoulli log-likelihood in float64
and its central finite differences."""
from __future__ import annotations

import numpy as np
import pytest
from scipy.sparse import coo_matrix
from scipy.sparse.csgraph import connected_components

import oracle


def cloud(seed=0, n=400, L=6.0):
    rng = np.random.default_rng(seed)
    clump = rng.standard_normal((n // 2, 3)) * 0.35 + L / 2
    p = np.concatenate([rng.random((n - n // 2, 3)) * L, clump]) % L
    return p.astype(np.float32), L


def test_fixed_sigmoid_is_the_logistic_and_monotone():
    t = np.linspace(-40, 40, 4001).astype(np.float32)
    s = np.array([oracle.sigmoid_fixed(float(x)) for x in t], np.float64)
    ref = 1.0 / (1.0 + np.exp(-np.clip(t.astype(np.float64), -30, 30)))
    assert np.abs(s - ref).max() <= 4e-7                      # degree-6 polynomial + float32 rounding
    assert np.all(np.diff(s) >= 0) and 0.0 < s[0] < 1e-12 and s[-1] == 1.0
    assert oracle.sigmoid_fixed(0.0) == 0.5


def test_rng_is_uniform_and_keyed_on_everything():
    u = np.array([oracle.rng_u24(7, 0, i, i + 1 + (i % 5)) for i in range(20000)], np.float64) / 2 ** 24
    assert abs(u.mean() - 0.5) < 4 * (1 / np.sqrt(12 * len(u)))
    hist = np.histogram(u, bins=16, range=(0, 1))[0]
    assert np.all(np.abs(hist - len(u) / 16) < 5 * np.sqrt(len(u) / 16))
    base = oracle.rng_u24(7, 0, 3, 9)
    assert len({base, oracle.rng_u24(8, 0, 3, 9), oracle.rng_u24(7, 1, 3, 9), oracle.rng_u24(7, 0, 4, 9),
                oracle.rng_u24(7, 0, 3, 10), oracle.rng_u24(7, 0, 9, 3)}) == 6


def test_large_alpha_reduces_to_deterministic_fof():
    """alpha -> infinity with b_cand = b: p = 1 inside b, so the sample IS the FoF graph."""
    p, L = cloud(1)
    b = 0.3
    lab, E = oracle.labels_brute(p, L, b)
    s = oracle.stochastic(p, L, b, b, 1e9, 5, 0, brute=True)
    # pairs at exactly d2 == b2 would have p = 1/2: none in this cloud
    assert s["n_edge"] == E and s["n_cand"] == E
    assert np.array_equal(s["labels"], lab)
    assert s["logp"] == 0.0


@pytest.mark.parametrize("sample", [0, 3])
def test_brute_equals_cells_and_scipy_components(sample):
    p, L = cloud(2, n=1500, L=8.0)
    a = oracle.stochastic(p, L, 0.5, 0.3, 4.0, 11, sample, brute=True)
    c = oracle.stochastic(p, L, 0.5, 0.3, 4.0, 11, sample)
    assert np.array_equal(a["labels"], c["labels"]) and a["n_cand"] == c["n_cand"] and a["n_edge"] == c["n_edge"]
    assert abs(a["logp"] - c["logp"]) <= 1e-9 * abs(a["logp"])
    assert np.abs(a["grad"] - c["grad"]).max() <= 1e-9 * np.abs(a["grad"]).max()
    ij, y, pr = oracle.stochastic_edges(p, L, 0.5, 0.3, 4.0, 11, sample)
    assert len(ij) == a["n_cand"] and y.sum() == a["n_edge"]
    e = ij[y == 1]
    n = len(p)
    _, comp = connected_components(coo_matrix((np.ones(len(e)), (e[:, 0], e[:, 1])), shape=(n, n)), directed=False)
    first = np.full(comp.max() + 1, n, np.int64)
    np.minimum.at(first, comp, np.arange(n))
    assert np.array_equal(a["labels"], first[comp].astype(np.int32))


def test_edge_frequencies_follow_p():
    """Over many samples every potential edge is kept with its own probability p (Eq. 8): binomial
    test per distance bin, and samples differ from each other."""
    p, L = cloud(3, n=300, L=5.0)
    S = 200
    ij, _, pr = oracle.stochastic_edges(p, L, 0.6, 0.4, 2.0, 99, 0)
    kept = np.zeros(len(ij))
    for s in range(S):
        ij_s, y, pr_s = oracle.stochastic_edges(p, L, 0.6, 0.4, 2.0, 99, s)
        assert np.array_equal(ij_s, ij) and np.array_equal(pr_s, pr)      # p does not depend on the sample
        kept += y
    order = np.argsort(pr)
    for chunk in np.array_split(order, 8):
        mean_p, var = pr[chunk].mean(), (pr[chunk] * (1 - pr[chunk])).sum() / S
        assert abs(kept[chunk].sum() / S - pr[chunk].sum()) <= 5 * np.sqrt(var) + 1e-9, mean_p
    assert 0 < kept.min() + 1 and kept.max() <= S and len(set(kept)) > 10


def test_logp_and_gradient_against_float64_bernoulli_likelihood():
    """log p(y) = sum y log p + (1 - y) log(1 - p) with the true logistic in float64, y frozen at the
    sampled edges; the oracle's analytic gradient against central differences of that function."""
    p32, L = cloud(4, n=120, L=4.0)
    bc, b, alpha = 0.7, 0.45, 3.0
    s = oracle.stochastic(p32, L, bc, b, alpha, 21, 2, brute=True)
    ij, y, pr = oracle.stochastic_edges(p32, L, bc, b, alpha, 21, 2)
    assert len(ij) > 200 and 0 < y.sum() < len(y)

    def loglik(x):
        d = x[ij[:, 0]] - x[ij[:, 1]]
        d -= L * np.round(d / L)
        t = alpha * (b * b - (d * d).sum(1)) / (b * b)
        return np.where(y == 1, -np.log1p(np.exp(-t)), -np.log1p(np.exp(t))).sum()

    x0 = p32.astype(np.float64)
    assert abs(s["logp"] - loglik(x0)) <= 2e-5 * abs(s["logp"])          # float32 p vs float64 logistic
    rng = np.random.default_rng(0)
    eps = 1e-6
    for i in rng.choice(np.unique(ij), size=10, replace=False):
        for ax in range(3):
            xp, xm = x0.copy(), x0.copy()
            xp[i, ax] += eps
            xm[i, ax] -= eps
            fd = (loglik(xp) - loglik(xm)) / (2 * eps)
            assert abs(fd - s["grad"][i, ax]) <= 2e-5 * max(1.0, np.abs(s["grad"]).max()), (i, ax, fd, s["grad"][i, ax])
    assert np.abs(s["grad"].sum(0)).max() <= 1e-9 * np.abs(s["grad"]).max() * len(p32)   # translation invariance
