"""Pins for the CPU oracle (oracle/fof_oracle.c) against things OTHER than itself:
hand cases (tests/golden), exact rational arithmetic, brute force, scipy library routines,
a float64 sandwich, closed forms and invariants.  CPU only.
"""
from fractions import Fraction

import numpy as np
import pytest
from scipy.sparse import coo_matrix
from scipy.sparse.csgraph import connected_components
from scipy.spatial import cKDTree

import oracle
from paper_2510_26851_b200 import inputs


def canon(component_of):
    """component ids -> label = minimum index in the component."""
    component_of = np.asarray(component_of)
    first = np.full(component_of.max() + 1, np.iinfo(np.int64).max)
    np.minimum.at(first, component_of, np.arange(len(component_of)))
    return first[component_of].astype(np.int32)


def same_partition(a, b):
    return np.array_equal(canon(np.unique(a, return_inverse=True)[1]), canon(np.unique(b, return_inverse=True)[1]))


def refines(fine, coarse):
    """every block of `fine` lies inside one block of `coarse`."""
    f = np.unique(fine, return_inverse=True)[1]
    rep = np.full(f.max() + 1, -1, dtype=np.int64)
    rep[f] = coarse
    return np.array_equal(rep[f], coarse)


# ------------------------------------------------------------------ wrap (oracle step 1)
def test_wrap_identity_and_edges():
    L = 8.0
    for x in (0.0, 0.5, 7.999999, np.nextafter(np.float32(8), np.float32(0))):
        assert oracle.wrap1(x, L) == float(np.float32(x))
    assert oracle.wrap1(8.0, L) == 0.0
    assert oracle.wrap1(-0.25, L) == 7.75
    assert oracle.wrap1(17.5, L) == 1.5
    assert oracle.wrap1(-16.0, L) == 0.0
    assert oracle.wrap1(-1e-12, L) == 0.0          # rounds to L, then the >= L guard
    rng = np.random.default_rng(1)
    x = (rng.standard_normal(2000) * 30).astype(np.float32)
    w = oracle.wrap(np.stack([x, x, x], 1), 3.7)[:, 0]
    assert (w >= 0).all() and (w < np.float32(3.7)).all()
    ref = np.mod(x.astype(np.float64), float(np.float32(3.7)))
    d = np.abs(w - ref)
    d = np.minimum(d, float(np.float32(3.7)) - d)
    assert d.max() < 1e-4                           # x mod L up to float32 rounding of x/L


def test_wrap_of_huge_coordinates_lands_in_the_box():
    """R6: beyond |x| ~ 2^24 L float32 cannot resolve L any more (x - L floor(x / L) is off by whole ulps of x); the
    result must still be a coordinate in [0, L), whatever it is (0 where even the +L fix-up does not reach)."""
    L = np.float32(3.7)
    x = np.array([-3e9, 3e9, -1e12, 1e12, -2.5e8, 7e10, -3.4e38, 3.4e38, -6.2e7, 6.2e7], dtype=np.float32)
    w = oracle.wrap(np.stack([x, x, x], 1), float(L))[:, 0]
    assert (w >= 0).all() and (w < L).all()
    # where float32 still resolves the box (|x| < 2^24 L = 6.2e7), the result is x mod L to rounding
    xs = np.array([-6.1e6, 6.1e6, -123456.7, 98765.4], dtype=np.float32)
    ws = oracle.wrap(np.stack([xs, xs, xs], 1), float(L))[:, 0]
    d = np.abs(ws - np.mod(xs.astype(np.float64), float(L)))
    assert np.minimum(d, float(L) - d).max() < 1.0    # off by at most an ulp of x (0.5 at 6e6)


def test_threaded_pair_search_equals_the_single_thread_oracle():
    """oracle.labels_cells_threads (the all-cores figure of bench.py) only changes the order in which edges reach the
    union-find: labels and E must be those of labels_cells, on clustered, uniform, tiny-grid and empty inputs."""
    rng = np.random.default_rng(12)
    w = inputs.scaled(inputs.CONFIGS["cfg1"], 24)
    cases = [(inputs.make_positions(w), w.L, w.b),
             ((rng.random((5000, 3)) * 10).astype(np.float32), 10.0, 0.35),
             ((rng.random((300, 3)) * 4).astype(np.float32), 4.0, 1.2),      # n = 3: every stencil wraps
             (np.zeros((0, 3), np.float32), 1.0, 0.1)]
    for p, L, b in cases:
        ref, E = oracle.labels_cells(p, L, b)
        for t in (1, 3, 8):
            got, Et = oracle.labels_cells_threads(p, L, b, t)
            assert np.array_equal(got, ref) and Et == E


def test_wrap_nonfinite_is_an_error():
    p = np.zeros((4, 3), np.float32)
    p[2, 1] = np.nan
    with pytest.raises(oracle.OracleError):
        oracle.labels_cells(p, 1.0, 0.1)
    p[2, 1] = np.inf
    with pytest.raises(oracle.OracleError):
        oracle.labels_brute(p, 1.0, 0.1)


# ------------------------------------------------------------------ predicate (oracle step 2)
def test_predicate_golden(golden_dir):
    n = 0
    for line in open(f"{golden_dir}/predicate_cases.txt"):
        if line.startswith("#") or not line.strip():
            continue
        L, b, xi, yi, zi, xj, yj, zj, exp = [float(t) for t in line.split()]
        assert oracle.link([xi, yi, zi], [xj, yj, zj], L, b) == bool(exp), line
        assert oracle.link([xj, yj, zj], [xi, yi, zi], L, b) == bool(exp), "symmetry: " + line
        n += 1
    assert n >= 20


def test_predicate_exact_on_dyadic_grid():
    """On a 2^-8 grid in a box L = 8 every float32 operation of the predicate is exact, so it
    must equal the mathematical statement evaluated in rational arithmetic."""
    rng = np.random.default_rng(2)
    L, q = 8, 256
    for b_num in (256, 300, 181):       # b = b_num / 256
        b = Fraction(b_num, q)
        for _ in range(1500):
            a = rng.integers(0, L * q, 3)
            d = rng.integers(-2 * b_num, 2 * b_num + 1, 3)
            c = (a + d) % (L * q)
            d2 = Fraction(0)
            for k in range(3):
                dd = Fraction(int(a[k]) - int(c[k]), q)
                if dd > Fraction(L, 2):
                    dd -= L
                elif dd < -Fraction(L, 2):
                    dd += L
                d2 += dd * dd
            got = oracle.link(a / q, c / q, L, float(b))
            assert got == (d2 <= b * b)


# ------------------------------------------------------------------ (a) brute force vs (b) cell list
def _adversarial(seed, L, b):
    """points on oracle-grid cell faces +-1 ulp, pairs at distance exactly b and b(1 +- 2^-23),
    points at 0 and at the largest float below L."""
    rng = np.random.default_rng(seed)
    n = int(np.floor(L / (b * (1 + 1e-6))))
    faces = (rng.integers(0, n, (300, 3)) * (L / n)).astype(np.float32)
    pts = [faces, np.nextafter(faces, np.float32(-1)), np.nextafter(faces, np.float32(2 * L))]
    base = (rng.random((200, 3)) * L).astype(np.float32)
    for f in (1.0, 1 - 2.0 ** -23, 1 + 2.0 ** -23):
        sh = base.copy()
        sh[:, rng.integers(0, 3)] += np.float32(b * f)
        pts += [base, sh]
    edge = np.array([[0, 0, 0], [np.nextafter(np.float32(L), np.float32(0))] * 3, [0, L / 2, 0]], np.float32)
    p = np.concatenate(pts + [edge]).astype(np.float32)
    p = np.mod(p, np.float32(L))
    p[p >= np.float32(L)] = 0
    return p[rng.permutation(len(p))]


@pytest.mark.parametrize("case", ["uniform", "clumps", "adversarial", "dense", "tiny_box"])
def test_brute_equals_cells(case):
    rng = np.random.default_rng(3)
    if case == "uniform":
        L, b = 1.0, 0.06
        p = rng.random((3000, 3)).astype(np.float32)
    elif case == "clumps":
        L, b = 1.0, 0.02
        w = inputs.Workload("t", 14, L, 0.2, 5, "clumps", halos=12, seed=5)
        p, b = inputs.make_positions(w), 0.02
    elif case == "adversarial":
        L, b = 8.0, 0.5
        p = _adversarial(4, L, b)
    elif case == "dense":
        L, b = 2.0, 0.11
        p = (rng.standard_normal((2500, 3)) * 0.15 + 1.0).astype(np.float32) % np.float32(L)
    else:  # fewer than 3 cells per axis: the cell-list path must fall back to all pairs
        L, b = 1.0, 0.4
        p = rng.random((300, 3)).astype(np.float32)
    la, Ea = oracle.labels_brute(p, L, b)
    lb, Eb = oracle.labels_cells(p, L, b)
    assert np.array_equal(la, lb)
    assert Ea == Eb


def test_labels_match_scipy_connected_components():
    """Library special case: edges from the predicate -> scipy csgraph -> min index per component."""
    rng = np.random.default_rng(6)
    L, b = 4.0, 0.45
    p = (rng.random((260, 3)) * L).astype(np.float32)
    N = len(p)
    w = oracle.wrap(p, L)
    ii, jj = [], []
    for i in range(N):
        for j in range(i + 1, N):
            if oracle.link(w[i], w[j], L, b):
                ii.append(i)
                jj.append(j)
    g = coo_matrix((np.ones(len(ii)), (ii, jj)), shape=(N, N))
    _, comp = connected_components(g, directed=False)
    expect = canon(comp)
    for fn in (oracle.labels_brute, oracle.labels_cells):
        lab, E = fn(p, L, b)
        assert np.array_equal(lab, expect)
        assert E == len(ii)


# ------------------------------------------------------------------ float64 sandwich at mid size
def _kd_labels(p, L, r):
    tree = cKDTree(p.astype(np.float64), boxsize=L)
    pairs = tree.query_pairs(r, output_type="ndarray")
    N = len(p)
    g = coo_matrix((np.ones(len(pairs)), (pairs[:, 0], pairs[:, 1])), shape=(N, N))
    return canon(connected_components(g, directed=False)[1]), len(pairs)


@pytest.mark.parametrize("name,n_side", [("cfg1", 40), ("cfg0", 32)])
def test_float64_sandwich(name, n_side):
    """Partition from the float32 oracle must be refined by the float64 partition at b(1-d) and
    must refine the one at b(1+d), d = 1e-5 + 8 * 2^-24 * L/b (float32 rounding of a wrapped
    difference is up to L * 2^-24 absolute)."""
    w = inputs.scaled(inputs.CONFIGS[name], n_side)
    p = inputs.make_positions(w)
    L, b = w.L, w.b
    lab, E = oracle.labels_cells(p, L, b)
    delta = 1e-5 + 8 * 2.0 ** -24 * (L / b)
    lo, E_lo = _kd_labels(p, L, b * (1 - delta))
    hi, E_hi = _kd_labels(p, L, b * (1 + delta))
    assert E_lo <= E <= E_hi
    assert refines(lo, lab) and refines(lab, hi)
    assert len(np.unique(lab)) < len(p)            # the case is not trivial


# ------------------------------------------------------------------ invariants
def _check_invariants(p, L, b, lab):
    N = len(p)
    idx = np.arange(N)
    assert (lab <= idx).all() and (lab >= 0).all()
    assert np.array_equal(lab[lab], lab)
    sizes = np.bincount(lab, minlength=N)
    assert sizes.sum() == N and (sizes[lab] > 0).all()


def test_invariants_and_connectivity():
    w = inputs.scaled(inputs.CONFIGS["cfg1"], 24)
    p = inputs.make_positions(w)
    L, b = w.L, w.b
    lab, E = oracle.labels_cells(p, L, b)
    _check_invariants(p, L, b, lab)
    # (1) every linked pair shares a label / (2) each group is connected — through an independent
    # float64 neighbour search for candidates, the oracle predicate for the decision
    tree = cKDTree(oracle.wrap(p, L).astype(np.float64), boxsize=L)
    cand = tree.query_pairs(b * 1.01, output_type="ndarray")
    wv = oracle.wrap(p, L)
    keep = np.array([oracle.link(wv[i], wv[j], L, b) for i, j in cand], dtype=bool)
    e = cand[keep]
    assert len(e) == E
    assert (lab[e[:, 0]] == lab[e[:, 1]]).all()
    g = coo_matrix((np.ones(len(e)), (e[:, 0], e[:, 1])), shape=(len(p), len(p)))
    ncomp, _ = connected_components(g, directed=False)
    assert ncomp == len(np.unique(lab))            # same count + (1) => groups are exactly the components


def test_permutation_invariance():
    w = inputs.scaled(inputs.CONFIGS["cfg1"], 20)
    p = inputs.make_positions(w)
    lab, E = oracle.labels_cells(p, w.L, w.b)
    perm = np.random.default_rng(7).permutation(len(p))
    lab2, E2 = oracle.labels_cells(p[perm], w.L, w.b)
    assert E == E2
    back = np.empty_like(lab2)
    back[perm] = lab2                               # labels of the permuted run, in original order
    assert same_partition(lab, back)
    # canonical label is the min index in the NEW numbering
    inv = np.empty_like(perm)
    inv[perm] = np.arange(len(perm))
    assert np.array_equal(lab2, canon(lab[perm]))


def test_translation_invariance_exact_shifts():
    """positions quantised to 2^-20 L with L a power of two; shifts are multiples of the quantum,
    so every difference is exact and the partition cannot change."""
    rng = np.random.default_rng(8)
    L, q = 4.0, 2.0 ** -18
    w = inputs.Workload("t", 16, L, 0.2, 5, "clumps", halos=10, seed=9)
    p = np.round(inputs.make_positions(w).astype(np.float64) / q) * q
    p = np.mod(p, L).astype(np.float32)
    b = 0.06
    lab, E = oracle.labels_cells(p, L, b)
    for _ in range(3):
        s = rng.integers(0, int(L / q), 3) * q
        ps = np.mod(p.astype(np.float64) + s, L).astype(np.float32)
        lab2, E2 = oracle.labels_cells(ps, L, b)
        assert E2 == E and np.array_equal(lab, lab2)


# ------------------------------------------------------------------ closed forms
def test_lattice_closed_form():
    n, L = 16, 16.0
    p = inputs.lattice(n, L)
    lab, E = oracle.labels_cells(p, L, 0.999)
    assert E == 0 and np.array_equal(lab, np.arange(n ** 3))
    lab, E = oracle.labels_cells(p, L, 1.0)          # <= is inclusive; links wrap the box
    assert E == 3 * n ** 3 and (lab == 0).all()
    lab_b, E_b = oracle.labels_brute(inputs.lattice(8, 4.0), 4.0, 0.5)
    assert (lab_b == 0).all() and E_b == 3 * 8 ** 3


def test_planted_cliques_closed_form():
    sizes = [1, 2, 3, 20, 21, 57, 300, 19, 5, 64]
    L, b = 64.0, 1.0
    p, ids = inputs.planted_cliques(10, sizes, L, b)
    lab, E = oracle.labels_cells(p, L, b)
    assert np.array_equal(lab, canon(ids))
    assert E == sum(s * (s - 1) // 2 for s in sizes)
    g = oracle.groups(p, lab, L, 20)
    assert sorted(g["group_size"].tolist()) == sorted(s for s in sizes if s >= 20)


def test_chain_closed_form():
    L = 32.0
    n = 64
    p = inputs.chain(n, L)                           # spacing 0.5
    lab, E = oracle.labels_cells(p, L, 0.5 / 0.9)    # spacing = 0.9 b -> one group around the box
    assert (lab == 0).all() and E == n
    lab, E = oracle.labels_cells(p, L, 0.5 / 1.1)    # spacing = 1.1 b -> singletons
    assert E == 0 and np.array_equal(lab, np.arange(n))
    lab_b, _ = oracle.labels_brute(p, L, 0.5 / 0.9)
    assert (lab_b == 0).all()


def test_poisson_edge_density(golden_dir):
    rng = np.random.default_rng(11)
    n_side, L = 60, 60.0
    p = (rng.random((n_side ** 3, 3)) * L).astype(np.float32)
    for line in open(f"{golden_dir}/poisson_edge_density.txt"):
        if line.startswith("#") or not line.strip():
            continue
        bf, e_over_n = [float(t) for t in line.split()]
        _, E = oracle.labels_cells(p, L, bf * L / n_side)
        mean = e_over_n * len(p)
        assert abs(E - mean) < 4 * np.sqrt(mean), (bf, E, mean)


# ------------------------------------------------------------------ groups
def test_groups_against_numpy():
    w = inputs.scaled(inputs.CONFIGS["cfg1"], 24)
    p = inputs.make_positions(w)
    m = inputs.make_masses(w)
    lab, _ = oracle.labels_cells(p, w.L, w.b)
    for N_min in (1, 2, 20):
        g = oracle.groups(p, lab, w.L, N_min, mass=m)
        u, cnt = np.unique(lab, return_counts=True)
        keep = cnt >= N_min
        assert g["K"] == keep.sum()
        assert np.array_equal(g["group_label"], u[keep])
        assert np.array_equal(g["group_size"], cnt[keep])
        msum = np.bincount(lab, weights=m.astype(np.float64), minlength=len(p))[u[keep]]
        assert np.allclose(g["group_mass"], msum, rtol=1e-12)
        lut = np.full(len(p), -1, np.int64)
        lut[u[keep]] = np.arange(keep.sum())
        assert np.array_equal(g["particle_group"], lut[lab])
        assert g["group_size"].sum() == (cnt[lab_to_idx(u, lab)] >= N_min).sum()
    g1 = oracle.groups(p, lab, w.L, 20)              # unit masses: mass == size exactly
    assert np.array_equal(g1["group_mass"], g1["group_size"].astype(np.float64))


def lab_to_idx(u, lab):
    return np.searchsorted(u, lab)


def test_com_equals_plain_mean_away_from_boundary():
    """Eq. 4: halo position = plain mean of member positions."""
    sizes = [30, 45, 25]
    L, b = 64.0, 1.0
    p, ids = inputs.planted_cliques(12, sizes, L, b)
    rng = np.random.default_rng(13)
    m = rng.uniform(0.5, 1.5, len(p)).astype(np.float32)
    lab, _ = oracle.labels_cells(p, L, b)
    g = oracle.groups(p, lab, L, 20, mass=m)
    for k, gl in enumerate(g["group_label"]):
        sel = lab == gl
        plain = np.average(p[sel].astype(np.float64), axis=0, weights=m[sel].astype(np.float64))
        assert np.allclose(g["group_com"][k], plain, atol=1e-9)
    gu = oracle.groups(p, lab, L, 20)
    for k, gl in enumerate(gu["group_label"]):
        assert np.allclose(gu["group_com"][k], p[lab == gl].astype(np.float64).mean(0), atol=1e-9)


def test_com_translates_across_the_boundary():
    L, b, q = 64.0, 1.0, 2.0 ** -16
    p, ids = inputs.planted_cliques(14, [40], L, b)
    p = (np.round(p.astype(np.float64) / q) * q).astype(np.float32)
    lab, _ = oracle.labels_cells(p, L, b)
    c0 = oracle.groups(p, lab, L, 20)["group_com"][0]
    for target in ([0.0, 0.0, 0.0], [L - 0.125, 0.25, L / 2]):
        s = np.round((np.array(target) - c0) / q) * q
        ps = np.mod(p.astype(np.float64) + s, L).astype(np.float32)
        lab2, _ = oracle.labels_cells(ps, L, b)
        assert np.array_equal(lab, lab2)
        c1 = oracle.groups(ps, lab2, L, 20)["group_com"][0]
        d = np.abs(np.mod(c0 + s, L) - c1)
        d = np.minimum(d, L - d)
        assert d.max() < 1e-9
    assert ((ps.max(0) - ps.min(0)) > L / 2).any()   # the last copy really straddles a face


def test_com_two_particles_straddling_a_face():
    L = 8.0
    p = np.array([[7.75, 1.0, 1.0], [0.25, 1.0, 3.0]], np.float32)
    lab, E = oracle.labels_brute(p, L, 3.0)
    assert E == 1 and (lab == 0).all()
    g = oracle.groups(p, lab, L, 2)
    assert np.allclose(g["group_com"][0], [0.0, 1.0, 2.0])
    g = oracle.groups(p, lab, L, 2, mass=np.array([3.0, 1.0], np.float32))
    assert np.allclose(g["group_com"][0], [7.875, 1.0, 1.5])
    assert np.allclose(g["group_mass"], [4.0])


def test_groups_edge_cases():
    g = oracle.groups(np.zeros((0, 3), np.float32), np.zeros(0, np.int32), 1.0, 20)
    assert g["K"] == 0
    lab, E = oracle.labels_cells(np.zeros((0, 3), np.float32), 1.0, 0.1)
    assert len(lab) == 0 and E == 0
    p = np.zeros((5, 3), np.float32)                 # coincident particles link (d = 0)
    lab, E = oracle.labels_cells(p, 1.0, 0.1)
    assert (lab == 0).all() and E == 10
    g = oracle.groups(p, lab, 1.0, 1)
    assert g["K"] == 1 and g["group_size"][0] == 5


# ------------------------------------------------------------------ Eq. 1 and P_ref
def test_linking_length_eq1():
    assert oracle.linking_length(0.2, 1000.0, 256 ** 3) == 0.78125
    assert oracle.linking_length(0.2, 1000.0, 128 ** 3) == 1.5625
    assert oracle.linking_length(0.2, 1.0, 32 ** 3) == float(np.float32(0.00625))
    for k, w in inputs.CONFIGS.items():
        assert oracle.linking_length(w.b_frac, w.L, w.N) == w.b, k


def test_pref_brute_force():
    rng = np.random.default_rng(15)
    L, b = 1.0, 0.1
    p = rng.random((500, 3)).astype(np.float32)
    n = int(np.floor(L / float(np.float32(b))))     # the oracle sees b rounded to float32: n = 9
    assert n == 9
    c = np.minimum(np.floor(p.astype(np.float64) * n / L).astype(int), n - 1)
    P = 0
    for i in range(len(p)):
        d = np.abs(c[i + 1:] - c[i])
        d = np.minimum(d, n - d)
        P += int((d.max(axis=1) <= 1).sum())
    assert oracle.pref(p, L, b) == P
