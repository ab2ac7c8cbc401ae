"""Parity of the CUDA path (through the C ABI) against the CPU oracle, element by element, on the
same seeded inputs.  Bars (BASELINE.json north_star): labels, group labels, sizes,
particle->group map and the edge count E bit-exact; masses within 1e-5 relative; periodic centre
of mass within 1e-5 * L per component.  Needs a B200: `pytest -m gpu`.
"""
import dataclasses

import numpy as np
import pytest

import oracle
from paper_2510_26851_b200 import inputs

pytestmark = pytest.mark.gpu

torch = pytest.importorskip("torch")


@pytest.fixture(scope="module")
def B():
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    from paper_2510_26851_b200 import binding

    binding.lib()  # fails loudly if libfof_b200.so is missing
    return binding


def gpu_fof(B, pos, L, b, N_min, mass=None, grid=None, particle_group=True, path="auto"):
    N = len(pos)
    f = B.FoF(N, L, b, N_min, grid=grid, path=path)
    dpos = torch.from_numpy(np.ascontiguousarray(pos, dtype=np.float32)).cuda().reshape(N, 3)
    dmass = None if mass is None else torch.from_numpy(mass).cuda()
    labels = f.link(dpos)
    status = f.status()
    E, tests, grid_pairs = f.link_stats()
    ran = f.link_path()
    g = f.groups(dpos, labels, mass=dmass, particle_group=particle_group)
    out = dict(labels=labels.cpu().numpy(), E=E, tests=tests, grid_pairs=grid_pairs, status=status, K=g["K"], grid=f.grid,
               ran=ran,
               group_label=g["group_label"].cpu().numpy(), group_size=g["group_size"].cpu().numpy(),
               group_mass=g["group_mass"].cpu().numpy(), group_com=g["group_com"].cpu().numpy(),
               particle_group=None if g["particle_group"] is None else g["particle_group"].cpu().numpy())
    f.close()
    return out


def check_against_oracle(B, pos, L, b, N_min, mass=None, grid=None, brute=False, paths=("cells", "blocks")):
    """Both implementations of H1-H5 (the block path where the plan admits it, and the cell path) against
    the oracle; returns the results of the last path in `paths` (the default one)."""
    lab, E = (oracle.labels_brute if brute else oracle.labels_cells)(pos, L, b)
    og = oracle.groups(pos, lab, L, N_min, mass=mass)
    for path in paths:
        got = _check_one(B, pos, L, b, N_min, mass, grid, path, lab, E, og)
    return got, lab, og


def _check_one(B, pos, L, b, N_min, mass, grid, path, lab, E, og):
    got = gpu_fof(B, pos, L, b, N_min, mass=mass, grid=grid, path=path)
    assert got["status"] == 0
    assert path != "cells" or got["ran"][0] == "cells"
    assert np.array_equal(got["labels"], lab), "canonical labels differ"
    assert got["E"] == E, "edge count differs"
    assert got["K"] == og["K"]
    assert np.array_equal(got["group_label"], og["group_label"])
    assert np.array_equal(got["group_size"], og["group_size"])
    assert np.array_equal(got["particle_group"], og["particle_group"])
    if og["K"]:
        assert np.all(np.abs(got["group_mass"] - og["group_mass"]) <= 1e-5 * og["group_mass"])
        if mass is None:
            assert np.array_equal(got["group_mass"], og["group_size"].astype(np.float32))
        d = np.abs(got["group_com"].astype(np.float64) - og["group_com"])
        d = np.minimum(d, float(np.float32(L)) - d)
        assert d.max() <= 1e-5 * L, f"centre of mass off by {d.max()}"
    return got


# --------------------------------------------------------------------------- closed forms, tiny
def test_lattice(B):
    n, L = 16, 16.0
    p = inputs.lattice(n, L)
    got = gpu_fof(B, p, L, 0.999, 1)
    assert got["E"] == 0 and np.array_equal(got["labels"], np.arange(n ** 3))
    assert got["K"] == n ** 3
    got = gpu_fof(B, p, L, 1.0, 20)
    assert got["E"] == 3 * n ** 3 and (got["labels"] == 0).all()
    assert got["K"] == 1 and got["group_size"][0] == n ** 3
    check_against_oracle(B, p, L, 1.0, 20)


def test_planted_cliques(B):
    sizes = [1, 2, 3, 20, 21, 57, 300, 19, 5, 64, 1000]
    L, b = 64.0, 1.0
    p, ids = inputs.planted_cliques(10, sizes, L, b)
    got, lab, _ = check_against_oracle(B, p, L, b, 20)
    assert got["E"] == sum(s * (s - 1) // 2 for s in sizes)
    assert sorted(got["group_size"].tolist()) == sorted(s for s in sizes if s >= 20)


def test_chain_wraps_the_box(B):
    L, n = 32.0, 64
    p = inputs.chain(n, L)
    got = gpu_fof(B, p, L, 0.5 / 0.9, 2)
    assert (got["labels"] == 0).all() and got["E"] == n
    got = gpu_fof(B, p, L, 0.5 / 1.1, 2)
    assert got["E"] == 0 and got["K"] == 0


@pytest.mark.parametrize("case", ["uniform", "adversarial", "dense", "unwrapped"])
def test_against_brute_force(B, case):
    rng = np.random.default_rng(3)
    if case == "uniform":
        L, b = 1.0, 0.06
        p = rng.random((3000, 3)).astype(np.float32)
    elif case == "adversarial":
        from test_oracle_pins import _adversarial

        L, b = 8.0, 0.5
        p = _adversarial(4, L, b)
    elif case == "dense":
        L, b = 2.0, 0.11
        p = (rng.standard_normal((2500, 3)) * 0.15 + 1.0).astype(np.float32) % np.float32(L)
    else:  # positions far outside [0, L): the wrap is part of the path
        L, b = 3.7, 0.2
        p = (rng.standard_normal((3000, 3)) * 9).astype(np.float32)
        p[:40] *= np.float32(1e9)   # and some beyond 2^24 L, where float32 no longer resolves the box (R6)
    for grid in (None, 3, "max"):
        if grid == "max":
            grid = int(np.floor(L / (float(np.float32(b)) * 1.001)))
        check_against_oracle(B, p, L, b, 5, brute=True, grid=grid)


def test_gpu_grid_cell_faces(B):
    """points on the faces of the GPU's own grids (+-1 ulp) and pairs at exactly b, b(1 +- 2^-23)."""
    rng = np.random.default_rng(21)
    L, b = 8.0, 0.5
    for n in (3, 7, 15):
        faces = (rng.integers(0, n, (400, 3)) * (L / n)).astype(np.float32)
        base = (rng.random((300, 3)) * L).astype(np.float32)
        sh = base.copy()
        sh[:100, 0] += np.float32(b)
        sh[100:200, 1] += np.float32(b * (1 + 2.0 ** -23))
        sh[200:, 2] += np.float32(b * (1 - 2.0 ** -23))
        p = np.concatenate([faces, np.nextafter(faces, np.float32(-1)), np.nextafter(faces, np.float32(99)),
                            base, sh]).astype(np.float32)
        p = np.mod(p, np.float32(L))
        p[p >= np.float32(L)] = 0
        check_against_oracle(B, p, L, b, 3, grid=n)


# --------------------------------------------------------------------------- BASELINE configs
def test_cfg0(B):
    w = inputs.CONFIGS["cfg0"]
    p = inputs.make_positions(w)
    got, lab, og = check_against_oracle(B, p, w.L, w.b, w.N_min)
    assert og["K"] > 10
    check_against_oracle(B, p, w.L, w.b, w.N_min, mass=inputs.make_masses(w))
    check_against_oracle(B, p, w.L, w.b, 1, grid=got["grid"][2])        # N_min = 1, tightest grid


def test_cfg1_scaled_several_grids(B):
    w = inputs.scaled(inputs.CONFIGS["cfg1"], 48)
    p = inputs.make_positions(w)
    m = inputs.make_masses(w)
    for grid in (None, 5, 100):
        check_against_oracle(B, p, w.L, w.b, w.N_min, mass=m, grid=grid)


def test_cfg1_full(B):
    w = inputs.CONFIGS["cfg1"]
    p = inputs.make_positions(w)
    got, lab, og = check_against_oracle(B, p, w.L, w.b, w.N_min)
    assert og["K"] > 10000
    check_against_oracle(B, p, w.L, w.b, w.N_min, mass=inputs.make_masses(w))


@pytest.mark.slow
def test_cfg2_full(B):
    """The headline workload (256^3), in the launch configuration bench.py times."""
    w = inputs.CONFIGS["cfg2"]
    p = inputs.make_positions(w)
    got, lab, og = check_against_oracle(B, p, w.L, w.b, w.N_min)
    assert og["K"] > 100000


def _full_size(B, name, paths=("auto",), min_edges=0, min_groups=0):
    """One BASELINE config (or stress stand-in) at FULL size through the whole path against the oracle; the
    Zel'dovich sets are generated with the FFTs on the GPU (same seeded white noise, same recipe)."""
    w = inputs.CONFIGS[name]
    p = inputs.make_positions(w, device="cuda")
    got, lab, og = check_against_oracle(B, p, w.L, w.b, w.N_min, paths=paths)
    assert got["E"] >= min_edges and og["K"] >= min_groups
    return got, lab, og


@pytest.mark.slow
@pytest.mark.parametrize("b_frac", ["0.1", "0.2", "0.3", "0.4"])
def test_cfg4_full_sweep(B, b_frac):
    """BASELINE.json configs[4] at full size (256^3, L = 2000, rms 1.0 spacing), every linking length of the
    sweep, both implementations of H1-H5.  As generated these sets hold E = 0 / 1 true edges (DESIGN.md
    section 4): they pin the fixed cost of the path (wrap, sort, cell walk, label scatter) bit for bit; the
    clustered regime of the sweep is test_stress_full below."""
    _full_size(B, "cfg4_b" + b_frac, paths=("cells", "blocks"))


@pytest.mark.slow
def test_cfg3_full(B):
    """BASELINE.json configs[3] at full size: 512^3 = 134 M particles (1.6 GB of positions, ~8 GB of host
    memory for the oracle)."""
    psutil = pytest.importorskip("psutil")
    if psutil.virtual_memory().available < 24 * 2 ** 30:
        pytest.skip("the 512^3 oracle needs ~8 GB of host memory on top of the input")
    if torch.cuda.mem_get_info()[0] < 24 * 2 ** 30:
        pytest.skip("not enough free device memory for the 512^3 workspace")
    _full_size(B, "cfg3")


@pytest.mark.slow
@pytest.mark.parametrize("name,min_edges,min_groups", [("stress_b0.2", 100000, 10), ("stress_b0.4", 1000000, 1000)])
def test_stress_full(B, name, min_edges, min_groups):
    """The stand-in for the "dense knots / giant component" intent of configs[3, 4] (same recipe past shell
    crossing, rms 4 spacings) at full size, element by element against the oracle:
    labels, E, sizes, masses, centres of mass, on both implementations of H1-H5."""
    got, lab, og = _full_size(B, name, paths=("cells", "blocks"), min_edges=min_edges, min_groups=min_groups)
    assert og["group_size"].max() >= 2 * inputs.CONFIGS[name].N_min


@pytest.mark.parametrize("b_frac", [0.1, 0.2, 0.3, 0.4])
def test_stress_scaled_sweep(B, b_frac):
    """The linking-length sweep of configs[4] on the shell-crossed recipe (rms 4 spacings) at 96^3: unlike the
    recipe as specified (E = 0 at this size) every point of the sweep has edges, from filaments (0.1) to a
    dominant component (0.4)."""
    w = dataclasses.replace(inputs.scaled(inputs.CONFIGS["stress_b0.2"], 96), b_frac=b_frac)
    p = inputs.make_positions(w)
    got, lab, og = check_against_oracle(B, p, w.L, w.b, w.N_min, mass=inputs.make_masses(w))
    assert got["E"] > 0


# --------------------------------------------------------------------------- stress: giant component, dense cells
def test_percolating_giant_component(B):
    """Poisson points at b = 1.0 x spacing (above the continuum percolation threshold ~0.87): one
    component holds most particles and wraps the box — stresses atomics, long parent chains and the
    centre of mass of a group wider than L/2."""
    rng = np.random.default_rng(31)
    n_side, L = 80, 80.0
    p = (rng.random((n_side ** 3, 3)) * L).astype(np.float32)
    got, lab, og = check_against_oracle(B, p, L, 1.0, 20, mass=rng.uniform(0.5, 1.5, len(p)).astype(np.float32))
    assert og["group_size"].max() > 0.5 * len(p)


def test_zeldovich_shell_crossing(B):
    """Zel'dovich recipe with the displacement pushed past shell crossing (rms 4 spacings): caustics,
    filaments and knots with cells holding many particles."""
    w = dataclasses.replace(inputs.scaled(inputs.CONFIGS["cfg4_b0.4"], 96), rms=4.0)
    p = inputs.make_positions(w)
    got, lab, og = check_against_oracle(B, p, w.L, w.b, w.N_min)
    assert og["K"] > 100


def test_one_dense_clump_many_per_cell(B):
    rng = np.random.default_rng(33)
    L, b = 100.0, 1.0
    clump = rng.standard_normal((20000, 3)) * 1.5 + 50.0
    bg = rng.random((20000, 3)) * L
    p = np.concatenate([bg, clump]).astype(np.float32) % np.float32(L)
    p = p[rng.permutation(len(p))]
    check_against_oracle(B, p, L, b, 20)


def test_block_path_falls_back_in_the_same_call(B):
    """The two ways the block path gives up, both decided on the device inside fof_link: (1) a block holds more
    records than a CTA keeps in shared memory (one clump of 20 000 in a few cells); (2) more linked ghosts than the
    equivalence list holds (blocks of 2 cells with b ~ the cell side: nearly every particle is a ghost of seven
    blocks).  Either way the cell path runs in the same call and the results are the oracle's."""
    rng = np.random.default_rng(35)
    clump = rng.standard_normal((20000, 3)) * 1.5 + 50.0
    bg = rng.random((20000, 3)) * 100.0
    p1 = (np.concatenate([bg, clump]) % 100.0).astype(np.float32)
    p2 = (rng.random((20000, 3)) * 10.0).astype(np.float32)
    for p, L, b in ((p1, 100.0, 1.0), (p2, 10.0, 1.0)):
        got, lab, og = check_against_oracle(B, p, L, b, 20, paths=("blocks",))
        assert got["ran"][1] > 0, "the plan should admit the block path"
        assert got["ran"][0] == "cells", "expected the fallback to the cell path"


@pytest.mark.parametrize("seed", range(24))
def test_random_small_boxes_both_paths(B, seed):
    """Differential test over random geometries: box side, linking length (so grids of 6 .. 45 cells per axis and
    block plans with 3 .. 12 blocks per axis, partial last blocks included), particle count NOT a multiple of 4,
    a mixture of uniform points, Gaussian clumps (some across the box faces), points exactly on cell faces and
    points outside [0, L).  Both implementations of H1-H5 against the oracle (brute force where it is cheap)."""
    rng = np.random.default_rng(1000 + seed)
    L = float(rng.choice([1.0, 7.3, 64.0, 1000.0]))
    n_cells = int(rng.integers(6, 46))
    b = float(np.float32(L / (n_cells + rng.uniform(0.05, 0.95)) / 1.001))
    N = int(rng.integers(300, 6000)) | 1
    n_cl = int(rng.integers(0, 6))
    parts = [rng.random((N, 3)) * L]
    for _ in range(n_cl):
        c = rng.random(3) * L
        if rng.random() < 0.5:
            c[rng.integers(0, 3)] = 0.0                       # a clump across a box face
        parts.append(c + rng.standard_normal((int(rng.integers(20, 400)), 3)) * b * rng.uniform(0.3, 2.0))
    faces = (rng.integers(0, n_cells, (60, 3)) * (L / n_cells)).astype(np.float64)   # on (or an ulp off) cell faces
    parts.append(faces + rng.choice([0.0, 1e-7 * L, -1e-7 * L], (60, 3)))
    p = np.concatenate(parts)
    p[:25] += L * rng.integers(-3, 4, (25, 3))                # outside the box: the wrap is part of the path
    p = p.astype(np.float32)
    p = p[rng.permutation(len(p))]
    mass = rng.uniform(0.5, 1.5, len(p)).astype(np.float32) if seed % 2 else None
    N_min = int(rng.choice([1, 2, 5, 20]))
    got, lab, og = check_against_oracle(B, p, L, b, N_min, mass=mass, brute=len(p) <= 2500)
    if seed % 3 == 0:                                         # and on a coarser grid than the plan's default
        check_against_oracle(B, p, L, b, N_min, mass=mass, grid=max(6, got["grid"][0] // 2))
    if seed % 3 == 1:                                         # and on the finest admissible grid (cell side ~ b)
        check_against_oracle(B, p, L, b, N_min, mass=mass, grid=got["grid"][2])


# --------------------------------------------------------------------------- invariants
def test_permutation_invariance_on_gpu(B):
    w = inputs.scaled(inputs.CONFIGS["cfg1"], 40)
    p = inputs.make_positions(w)
    a = gpu_fof(B, p, w.L, w.b, w.N_min)
    perm = np.random.default_rng(41).permutation(len(p))
    c = gpu_fof(B, p[perm], w.L, w.b, w.N_min)
    assert a["E"] == c["E"] and a["K"] == c["K"]
    assert sorted(a["group_size"].tolist()) == sorted(c["group_size"].tolist())
    # partition identical: the canonical particle of the permuted run, expressed in ORIGINAL numbering, names the
    # same blocks; both sides relabelled to the minimum original index of the block must be equal arrays
    back = np.empty_like(c["labels"])
    back[perm] = perm[c["labels"]]
    canon = np.full(len(p), len(p), dtype=np.int64)
    np.minimum.at(canon, back, np.arange(len(p)))
    assert np.array_equal(canon[back], a["labels"])


def test_repeatable(B):
    """Three runs of the same input: labels, E and sizes identical; masses and centres of mass (summed with
    float atomics, so order dependent) within the parity tolerance of each other."""
    w = inputs.CONFIGS["cfg0"]
    p = inputs.make_positions(w)
    m = inputs.make_masses(w)
    runs = [gpu_fof(B, p, w.L, w.b, w.N_min, mass=m) for _ in range(3)]
    for r in runs[1:]:
        assert np.array_equal(r["labels"], runs[0]["labels"]) and r["E"] == runs[0]["E"]
        assert np.array_equal(r["group_size"], runs[0]["group_size"])
        assert np.all(np.abs(r["group_mass"] - runs[0]["group_mass"]) <= 1e-5 * runs[0]["group_mass"])
        d = np.abs(r["group_com"].astype(np.float64) - runs[0]["group_com"])
        assert np.minimum(d, w.L - d).max() <= 1e-5 * w.L


@pytest.mark.parametrize("members", [4000, 4095, 4096, 9000])
def test_mass_com_worst_case_of_the_float32_atomics(B, members):
    """group_reduce_kernel sums groups of fewer than 4096 members with float32 atomics.
    Worst case for that branch: one group of ~4000 members with masses U(0.5, 1.5), a chain more than 10 b
    (here ~L/3) long that crosses a box face, so the deltas are large and of one sign; 4096 and 9000 members
    take the float64 branch on the same geometry.  Mass within 1e-5 relative, centre of mass within 1e-5 L."""
    rng = np.random.default_rng(77 + members)
    L, b = 64.0, 0.05
    x = (np.arange(members) * (0.9 * b * 0.1) + 0.97 * L) % L      # spacing 0.09 b: 4000 members span 18 = 360 b
    chainp = np.stack([x, np.full(members, 20.0) + rng.uniform(-0.2 * b, 0.2 * b, members),
                       np.full(members, 31.0) + rng.uniform(-0.2 * b, 0.2 * b, members)], 1)
    bg = rng.random((3000, 3)) * L
    p = np.concatenate([chainp, bg]).astype(np.float32)
    p[p >= np.float32(L)] = 0.0
    p = p[rng.permutation(len(p))]
    mass = rng.uniform(0.5, 1.5, len(p)).astype(np.float32)
    for _ in range(3):   # the summation order changes from run to run
        got, lab, og = check_against_oracle(B, p, L, b, 20, mass=mass)
    assert og["group_size"].max() >= members


# --------------------------------------------------------------------------- edge cases and errors
def test_empty_and_tiny(B):
    got = gpu_fof(B, np.zeros((0, 3), np.float32), 1.0, 0.1, 20)
    assert got["K"] == 0 and got["E"] == 0 and len(got["labels"]) == 0
    got = gpu_fof(B, np.array([[0.5, 0.5, 0.5]], np.float32), 1.0, 0.1, 1)
    assert got["K"] == 1 and got["labels"][0] == 0 and got["group_size"][0] == 1
    assert np.allclose(got["group_com"][0], 0.5)
    p = np.zeros((5, 3), np.float32)                    # coincident particles link (d = 0)
    got = gpu_fof(B, p, 1.0, 0.1, 1)
    assert (got["labels"] == 0).all() and got["E"] == 10 and got["group_size"][0] == 5


def test_nonfinite_sets_status(B):
    p = np.random.default_rng(5).random((1000, 3)).astype(np.float32)
    p[17, 1] = np.nan
    got = gpu_fof(B, p, 1.0, 0.05, 20)
    assert got["status"] == B.FOF_ERR_NONFINITE
    p[17, 1] = np.inf
    assert gpu_fof(B, p, 1.0, 0.05, 20)["status"] == B.FOF_ERR_NONFINITE


def test_capacity_error(B):
    sizes = [30] * 8
    p, _ = inputs.planted_cliques(10, sizes, 64.0, 1.0)
    f = B.FoF(len(p), 64.0, 1.0, 20)
    dpos = torch.from_numpy(p).cuda()
    labels = f.link(dpos)
    out = f.alloc_groups(cap=4)
    with pytest.raises(B.FofError) as e:
        f.groups(dpos, labels, out=out)
    assert e.value.code == B.FOF_ERR_CAPACITY
    g = f.groups(dpos, labels)
    assert g["K"] == 8


def test_groups_is_stateless_on_given_labels(B):
    """fof_groups works from (pos, labels) alone — here labels from the oracle, fresh workspace."""
    w = inputs.scaled(inputs.CONFIGS["cfg1"], 32)
    p = inputs.make_positions(w)
    lab, _ = oracle.labels_cells(p, w.L, w.b)
    og = oracle.groups(p, lab, w.L, w.N_min)
    f = B.FoF(len(p), w.L, w.b, w.N_min)
    g = f.groups(torch.from_numpy(p).cuda(), torch.from_numpy(lab).cuda(), particle_group=True)
    assert g["K"] == og["K"]
    assert np.array_equal(g["group_size"].cpu().numpy(), og["group_size"])
    assert np.array_equal(g["particle_group"].cpu().numpy(), og["particle_group"])


def test_run_host_path(B):
    """The host-buffer entry point (what bench.py's e2e leg times) gives the same answer."""
    w = inputs.scaled(inputs.CONFIGS["cfg1"], 48)
    p = inputs.make_positions(w)
    m = inputs.make_masses(w)
    lab, _ = oracle.labels_cells(p, w.L, w.b)
    og = oracle.groups(p, lab, w.L, w.N_min, mass=m)
    N = len(p)
    h = B.fof_create(N, w.L, w.b, w.N_min)
    cap = N // w.N_min
    dev = torch.empty(B.fof_host_device_bytes(h, cap) + 256, dtype=torch.uint8, device="cuda")
    hp = torch.from_numpy(p).pin_memory()
    hm = torch.from_numpy(m).pin_memory()
    hl = torch.empty(N, dtype=torch.int32).pin_memory()
    gl = torch.empty(cap, dtype=torch.int32).pin_memory()
    gs = torch.empty(cap, dtype=torch.int32).pin_memory()
    gm = torch.empty(cap, dtype=torch.float32).pin_memory()
    gc = torch.empty((cap, 3), dtype=torch.float32).pin_memory()
    pg = torch.empty(N, dtype=torch.int32).pin_memory()
    K = B.fof_run_host(h, hp, hm, hl, gl, gs, gm, gc, pg, cap, dev)
    assert K == og["K"]
    assert np.array_equal(hl.numpy(), lab)
    assert np.array_equal(gs.numpy()[:K], og["group_size"])
    assert np.array_equal(pg.numpy(), og["particle_group"])
    assert np.all(np.abs(gm.numpy()[:K] - og["group_mass"]) <= 1e-5 * og["group_mass"])
    d = np.abs(gc.numpy()[:K].astype(np.float64) - og["group_com"])
    assert np.minimum(d, w.L - d).max() <= 1e-5 * w.L
    B.fof_destroy(h)


def test_host_pipeline_against_oracle(B):
    """fof_host_submit / fof_host_wait: six different inputs through the two slots, two in flight all the time;
    every result equals the oracle's for ITS input (a mixed-up slot, a copy that overtakes its kernel or a result
    read before its copy landed would show), for both link paths."""
    import dataclasses
    base = inputs.scaled(inputs.CONFIGS["cfg1"], 40)
    ws = [dataclasses.replace(base, seed=base.seed + 100 * k) for k in range(6)]
    ps = [inputs.make_positions(w) for w in ws]
    N = len(ps[0])
    assert all(len(p) == N for p in ps)
    ms = [inputs.make_masses(w) for w in ws]
    want = []
    for p, m in zip(ps, ms):
        lab, _ = oracle.labels_cells(p, base.L, base.b)
        want.append((lab, oracle.groups(p, lab, base.L, base.N_min, mass=m)))
    assert len({o["K"] for _, o in want}) > 1  # the inputs really differ
    cap = N // base.N_min
    pin = lambda *s, dt=torch.int32: torch.empty(*s, dtype=dt).pin_memory()  # noqa: E731
    for path in ("cells", "blocks"):
        h = B.fof_create(N, base.L, base.b, base.N_min)
        B.fof_set_path(h, {"cells": B.FOF_PATH_CELLS, "blocks": B.FOF_PATH_BLOCKS}[path])
        nbytes = B.fof_host_device_bytes(h, cap) + 256
        dev = [torch.empty(nbytes, dtype=torch.uint8, device="cuda") for _ in range(2)]
        hp = [torch.from_numpy(p).pin_memory() for p in ps]
        hm = [torch.from_numpy(m).pin_memory() for m in ms]
        outs = [dict(hl=pin(N), gl=pin(cap), gs=pin(cap), gm=pin(cap, dt=torch.float32),
                     gc=pin((cap, 3), dt=torch.float32), pg=pin(N)) for _ in range(2)]

        def submit(k):
            o = outs[k % 2]
            for t in o.values():
                t.fill_(-7)
            B.fof_host_submit(h, k % 2, hp[k], hm[k], o["hl"], o["gl"], o["gs"], o["gm"], o["gc"], o["pg"], cap,
                              dev[k % 2])

        def collect(k):
            o = outs[k % 2]
            K = B.fof_host_wait(h, k % 2)
            lab, og = want[k]
            assert K == og["K"], (path, k)
            assert np.array_equal(o["hl"].numpy(), lab), (path, k)
            assert np.array_equal(o["gs"].numpy()[:K], og["group_size"])
            assert np.array_equal(o["gl"].numpy()[:K], og["group_label"])
            assert np.array_equal(o["pg"].numpy(), og["particle_group"])
            assert np.all(np.abs(o["gm"].numpy()[:K] - og["group_mass"]) <= 1e-5 * og["group_mass"])
            d = np.abs(o["gc"].numpy()[:K].astype(np.float64) - og["group_com"])
            assert np.minimum(d, base.L - d).max() <= 1e-5 * base.L

        submit(0)
        for k in range(1, len(ps)):
            submit(k)
            collect(k - 1)
        collect(len(ps) - 1)
        B.fof_destroy(h)


def test_host_pipeline_errors(B):
    """Call-order and deferred errors of the pipelined host path."""
    w = inputs.scaled(inputs.CONFIGS["cfg1"], 24)
    p = inputs.make_positions(w)
    N = len(p)
    lab, _ = oracle.labels_cells(p, w.L, w.b)
    og = oracle.groups(p, lab, w.L, w.N_min)
    assert og["K"] >= 2
    h = B.fof_create(N, w.L, w.b, w.N_min)
    cap = N // w.N_min
    dev = torch.empty(B.fof_host_device_bytes(h, cap) + 256, dtype=torch.uint8, device="cuda")
    pin = lambda *s, dt=torch.int32: torch.empty(*s, dtype=dt).pin_memory()  # noqa: E731
    hp, hl = torch.from_numpy(p).pin_memory(), pin(N)
    gl, gs, gm, gc = pin(cap), pin(cap), pin(cap, dt=torch.float32), pin((cap, 3), dt=torch.float32)
    with pytest.raises(B.FofError) as e:
        B.fof_host_wait(h, 0)  # nothing submitted
    assert e.value.code == B.FOF_ERR_STATE
    with pytest.raises(B.FofError) as e:
        B.fof_host_submit(h, 2, hp, None, hl, gl, gs, gm, gc, None, cap, dev)
    assert e.value.code == B.FOF_ERR_INVALID_ARG
    B.fof_host_submit(h, 0, hp, None, hl, gl, gs, gm, gc, None, cap, dev)
    with pytest.raises(B.FofError) as e:
        B.fof_host_submit(h, 0, hp, None, hl, gl, gs, gm, gc, None, cap, dev)  # slot busy
    assert e.value.code == B.FOF_ERR_STATE
    assert B.fof_host_wait(h, 0) == og["K"]
    assert np.array_equal(hl.numpy(), lab)
    with pytest.raises(B.FofError) as e:
        B.fof_host_wait(h, 0)  # already collected
    assert e.value.code == B.FOF_ERR_STATE
    # more groups than capacity: K is reported, the labels still arrive
    small = og["K"] - 1
    dev2 = torch.empty(B.fof_host_device_bytes(h, small) + 256, dtype=torch.uint8, device="cuda")
    hl.fill_(-1)
    B.fof_host_submit(h, 1, hp, None, hl, gl, gs, gm, gc, None, small, dev2)
    with pytest.raises(B.FofError) as e:
        B.fof_host_wait(h, 1)
    assert e.value.code == B.FOF_ERR_CAPACITY
    assert np.array_equal(hl.numpy(), lab)
    # a non-finite coordinate is reported by the wait
    bad = torch.from_numpy(p.copy()).pin_memory()
    bad[5, 1] = float("nan")
    B.fof_host_submit(h, 0, bad, None, hl, gl, gs, gm, gc, None, cap, dev)
    with pytest.raises(B.FofError) as e:
        B.fof_host_wait(h, 0)
    assert e.value.code == B.FOF_ERR_NONFINITE
    # the slot is usable again, and destroying the handle with a submit in flight is safe
    B.fof_host_submit(h, 0, hp, None, hl, gl, gs, gm, gc, None, cap, dev)
    B.fof_destroy(h)
    torch.cuda.synchronize()


@pytest.mark.parametrize("N", [0, 1, 5])
def test_host_calls_on_empty_and_tiny_inputs(B, N):
    """fof_run_host and fof_host_submit / fof_host_wait with no particle, one particle, five coincident ones."""
    p = np.full((N, 3), 0.5, np.float32)
    h = B.fof_create(N, 1.0, 0.1, 1)
    cap = max(N, 1)
    pin = lambda *s, dt=torch.int32: torch.empty(*s, dtype=dt).pin_memory()  # noqa: E731
    hp = torch.from_numpy(p).pin_memory() if N else torch.zeros((1, 3)).pin_memory()
    hl, gl, gs, pg = pin(cap), pin(cap), pin(cap), pin(cap)
    gm, gc = pin(cap, dt=torch.float32), pin((cap, 3), dt=torch.float32)
    dev = [torch.empty(B.fof_host_device_bytes(h, cap) + 256, dtype=torch.uint8, device="cuda") for _ in range(2)]

    def check(K):
        assert K == (1 if N else 0)
        if N:
            assert (hl.numpy()[:N] == 0).all() and gs.numpy()[0] == N and gl.numpy()[0] == 0
            assert (pg.numpy()[:N] == 0).all() and abs(gm.numpy()[0] - N) < 1e-6
            assert np.allclose(gc.numpy()[0], 0.5)

    for t in (hl, gl, gs, pg):
        t.fill_(-3)
    check(B.fof_run_host(h, hp, None, hl, gl, gs, gm, gc, pg, cap, dev[0]))
    for slot in (0, 1, 0):
        for t in (hl, gl, gs, pg):
            t.fill_(-3)
        B.fof_host_submit(h, slot, hp, None, hl, gl, gs, gm, gc, pg, cap, dev[slot])
        check(B.fof_host_wait(h, slot))
    B.fof_destroy(h)


@pytest.mark.parametrize("n_particles", [4099, 65537])
def test_unaligned_caller_pointers(B, n_particles):
    """pos / labels / particle_group that are only 4-byte aligned (views one element into a buffer) and
    an N that is not a multiple of 4: the kernels must take their scalar load/store paths."""
    rng = np.random.default_rng(77)
    L, b, N_min = 50.0, 1.0, 3
    N = n_particles
    clump = rng.standard_normal((N // 3, 3)) * 0.8 + 25.0
    p = np.concatenate([rng.random((N - N // 3, 3)) * L, clump]).astype(np.float32) % np.float32(L)
    p = p[rng.permutation(N)]
    m = rng.uniform(0.5, 1.5, N).astype(np.float32)
    lab, E = oracle.labels_cells(p, L, b)
    og = oracle.groups(p, lab, L, N_min, mass=m)

    f = B.FoF(N, L, b, N_min)
    buf_p = torch.empty(3 * N + 1, dtype=torch.float32, device="cuda")
    dpos = buf_p[1:].view(N, 3)
    dpos.copy_(torch.from_numpy(p))
    buf_l = torch.empty(N + 1, dtype=torch.int32, device="cuda")
    labels = buf_l[1:]
    buf_g = torch.empty(N + 3, dtype=torch.int32, device="cuda")
    pg = buf_g[3:]
    buf_m = torch.empty(N + 1, dtype=torch.float32, device="cuda")
    dm = buf_m[1:]
    dm.copy_(torch.from_numpy(m))
    assert dpos.data_ptr() % 16 == 4 and labels.data_ptr() % 16 == 4 and pg.data_ptr() % 16 == 12
    B.fof_link(f.h, dpos, labels, f.ws)
    assert f.status() == 0
    assert np.array_equal(labels.cpu().numpy(), lab)
    assert f.link_stats()[0] == E
    out = f.alloc_groups()
    K = B.fof_groups(f.h, dpos, dm, labels, f.ws, out["group_label"], out["group_size"], out["group_mass"],
                     out["group_com"], pg, out["cap"])
    assert K == og["K"]
    assert np.array_equal(out["group_size"][:K].cpu().numpy(), og["group_size"])
    assert np.array_equal(pg.cpu().numpy(), og["particle_group"])
    gm = out["group_mass"][:K].cpu().numpy()
    assert np.all(np.abs(gm - og["group_mass"]) <= 1e-5 * og["group_mass"])
    d = np.abs(out["group_com"][:K].cpu().numpy().astype(np.float64) - og["group_com"])
    assert np.minimum(d, L - d).max() <= 1e-5 * L
    f.close()


# --------------------------------------------------------------------------- NEXT-1: decoration + backward
@pytest.mark.parametrize("weighted", [False, True])
def test_sigma_and_backward_against_oracle(B, weighted):
    """fof_group_sigma / fof_groups_backward (section 3.1 Eq. 4, 3.1.1 Eq. 5) on a clustered set
    with groups that cross the box faces.  Tolerances: the CUDA path reads the float32 group_com /
    group_mass / group_sigma that fof_groups / fof_group_sigma wrote (rounded once, <= ulp/2), the
    oracle its own float64 values; a shift e of the centre changes sigma^2 by |e|^2 only (sum m delta
    = 0), so sigma agrees to float32 rounding; in the backward, delta / sigma inherits
    |e| / sigma <= ulp(L) / sigma per axis."""
    w = inputs.scaled(inputs.CONFIGS["cfg1"], 48)
    p = inputs.make_positions(w)
    m = inputs.make_masses(w) if weighted else None
    lab, _ = oracle.labels_cells(p, w.L, w.b)
    og = oracle.groups(p, lab, w.L, w.N_min, mass=m)
    osig = oracle.group_sigma(p, og["particle_group"], w.L, og["group_com"], mass=m)
    rng = np.random.default_rng(8)
    K = og["K"]
    assert K > 50
    G = rng.standard_normal((K, 3)).astype(np.float32)
    C = rng.standard_normal(K).astype(np.float32)
    ograd = oracle.groups_backward(p, og["particle_group"], w.L, og["group_mass"], og["group_com"], G,
                                   group_sigma=osig, grad_sigma=C, mass=m)
    ograd_x = oracle.groups_backward(p, og["particle_group"], w.L, og["group_mass"], og["group_com"], G, mass=m)

    f = B.FoF(len(p), w.L, w.b, w.N_min)
    dpos = torch.from_numpy(p).cuda()
    dm = None if m is None else torch.from_numpy(m).cuda()
    labels = f.link(dpos)
    g = f.groups(dpos, labels, mass=dm, particle_group=True)
    assert g["K"] == K
    sig = f.group_sigma(dpos, g, mass=dm)
    s_gpu = sig.cpu().numpy().astype(np.float64)
    assert np.all(np.abs(s_gpu - osig) <= 2e-6 * osig + 1e-7 * w.L)
    dG, dC = torch.from_numpy(G).cuda(), torch.from_numpy(C).cuda()
    gx = f.groups_backward(dpos, g, grad_com=dG, mass=dm).cpu().numpy().astype(np.float64)
    assert np.abs(gx - ograd_x).max() <= 2e-6 * np.abs(ograd_x).max()
    assert (gx[og["particle_group"] < 0] == 0).all()
    gall = f.groups_backward(dpos, g, grad_com=dG, group_sigma=sig, grad_sigma=dC, mass=dm).cpu().numpy().astype(np.float64)
    ulp_L = float(np.spacing(np.float32(w.L)))
    pg = og["particle_group"]
    member = pg >= 0
    mm = np.ones(len(p)) if m is None else m.astype(np.float64)
    wgt = np.zeros(len(p))
    wgt[member] = mm[member] / og["group_mass"][pg[member]]
    bound = np.zeros(len(p))
    bound[member] = 4e-6 * np.abs(ograd).max() + 2.0 * np.abs(C[pg[member]]) * wgt[member] * ulp_L / osig[pg[member]]
    assert np.all(np.abs(gall - ograd).max(1) <= bound + 1e-30)
    f.close()


def test_backward_without_groups_is_zero(B):
    rng = np.random.default_rng(12)
    p = (rng.random((5000, 3)) * 100.0).astype(np.float32)   # sparse: no group reaches N_min
    f = B.FoF(len(p), 100.0, 0.5, 20)
    dpos = torch.from_numpy(p).cuda()
    g = f.groups(dpos, f.link(dpos), particle_group=True)
    assert g["K"] == 0
    assert f.group_sigma(dpos, g).numel() == 0
    assert (f.groups_backward(dpos, g) == 0).all()
    f.close()


@pytest.mark.parametrize("grid", [600, 1024])
def test_large_grids_take_the_wide_bin_paths(B, grid):
    """n = 600 (2.2e8 cells: bins of 2^13 cells) and n = 1024 (2^30 cells: bins of 2^15 cells, 128 KB of
    shared-memory counters per CTA): the sort's wide-bin configurations, far more cells than particles."""
    rng = np.random.default_rng(91)
    L, b, N_min = 2000.0, 1.0, 5
    bg = rng.random((150000, 3)) * L
    centres = rng.random((300, 3)) * L
    clumps = (centres[:, None, :] + rng.standard_normal((300, 40, 3)) * 0.6).reshape(-1, 3)
    p = (np.concatenate([bg, clumps]) % L).astype(np.float32)
    p[p >= np.float32(L)] = 0.0
    p = p[rng.permutation(len(p))]
    got, lab, og = check_against_oracle(B, p, L, b, N_min, grid=grid)
    assert got["grid"][0] == grid and og["K"] >= 250


# --------------------------------------------------------------------------- NEXT-3: stochastic-edge FoF
@pytest.mark.parametrize("alpha,kappa", [(5.0, 1.5), (0.5, 1.25), (50.0, 1.0)])
def test_stochastic_link_against_oracle(B, alpha, kappa):
    """fof_link_stochastic (section 3.2 Eq. 8): labels of every sample and the numbers of potential and
    sampled edges bit-exact (both sides take u < p on identical float32 bits), log p(y) to float64
    summation order, the score function to float32 accumulation (warp scans, another order than the oracle's)."""
    w = inputs.scaled(inputs.CONFIGS["cfg1"], 40)
    p = inputs.make_positions(w)
    b_link = w.b
    b_cand = float(np.float32(kappa * w.b))
    f = B.FoF(len(p), w.L, b_cand, w.N_min, path="cells")
    dpos = torch.from_numpy(p).cuda()
    f.link(dpos)                                   # the binning every sample re-uses
    for sample in (0, 1, 7):
        o = oracle.stochastic(p, w.L, b_cand, b_link, alpha, 1234, sample)
        labels, logp, grad = f.link_stochastic(b_link, alpha, 1234, sample)
        E, ncand, _ = f.link_stats()
        assert ncand == o["n_cand"] and E == o["n_edge"]
        assert np.array_equal(labels.cpu().numpy(), o["labels"]), "sampled components differ"
        assert abs(float(logp.item()) - o["logp"]) <= 2e-6 * abs(o["logp"]) + 1e-6   # float32 log terms
        g = grad.cpu().numpy().astype(np.float64)
        assert np.abs(g - o["grad"]).max() <= 2e-5 * np.abs(o["grad"]).max()
    # samples differ from each other, and a different seed gives a different graph
    a, logp_a, grad_a = f.link_stochastic(b_link, alpha, 1234, 0, want_grad=False)
    # without the score function only the owning side of each pair is evaluated: same sample, same numbers
    o0 = oracle.stochastic(p, w.L, b_cand, b_link, alpha, 1234, 0)
    E, ncand, _ = f.link_stats()
    assert grad_a is None and ncand == o0["n_cand"] and E == o0["n_edge"]
    assert np.array_equal(a.cpu().numpy(), o0["labels"])
    assert abs(float(logp_a.item()) - o0["logp"]) <= 2e-6 * abs(o0["logp"]) + 1e-6
    c = f.link_stochastic(b_link, alpha, 1235, 0, want_grad=False)[0]
    assert alpha >= 50.0 or not torch.equal(a, c)
    f.close()


@pytest.mark.parametrize("S,drop", [(1, 0), (4, 0), (7, 0), (7, 1), (7, 2), (7, 3)])
def test_stochastic_batch_equals_single_samples_and_oracle(B, S, drop):
    """fof_link_stochastic_batch: sample k of the batch = fof_link_stochastic(sample0 + k) = the oracle's sample
    (labels and edge counts bit-exact, log p and score function to summation order); S = 7 mixes a pass of four
    samples with single ones.  drop = 1, 2, 3: N % 4 != 0, so the per-sample union-find arrays rel_s + k N are
    not 16-byte aligned (write_labels_kernel then takes its scalar path)."""
    w = inputs.scaled(inputs.CONFIGS["cfg1"], 40)
    p = inputs.make_positions(w)
    p = np.ascontiguousarray(p[:len(p) - drop]) if drop else p
    assert len(p) % 4 == (4 - drop) % 4
    b_link, alpha = w.b, 4.0
    b_cand = float(np.float32(1.5 * w.b))
    f = B.FoF(len(p), w.L, b_cand, w.N_min, path="cells")
    f.link(torch.from_numpy(p).cuda())
    labels, logp, grad = f.link_stochastic_batch(b_link, alpha, 99, 3, S)
    E_all, ncand, _ = f.link_stats()
    E_sum = 0
    for k in range(S):
        o = oracle.stochastic(p, w.L, b_cand, b_link, alpha, 99, 3 + k)
        assert ncand == o["n_cand"]
        E_sum += o["n_edge"]
        assert np.array_equal(labels[k].cpu().numpy(), o["labels"]), f"sample {k}: components differ"
        assert abs(float(logp[k].item()) - o["logp"]) <= 2e-6 * abs(o["logp"]) + 1e-6
        gk = grad[k].cpu().numpy().astype(np.float64)
        assert np.abs(gk - o["grad"]).max() <= 2e-5 * np.abs(o["grad"]).max()
        l1, lp1, g1 = f.link_stochastic(b_link, alpha, 99, 3 + k)
        assert torch.equal(l1, labels[k])
        assert abs(float(lp1.item()) - float(logp[k].item())) <= 2e-6 * abs(o["logp"]) + 1e-6
    assert E_all == E_sum
    # without the score function
    labels2, logp2, grad2 = f.link_stochastic_batch(b_link, alpha, 99, 3, S, want_grad=False)
    assert grad2 is None and torch.equal(labels2, labels)
    assert torch.allclose(logp2, logp, rtol=2e-6, atol=1e-6)
    f.close()


@pytest.mark.parametrize("alpha,kappa,S,drop", [(5.0, 1.5, 7, 0), (0.5, 1.25, 4, 1), (50.0, 1.0, 1, 2), (4.0, 1.5, 5, 3)])
def test_stochastic_list_against_oracle(B, alpha, kappa, S, drop):
    """fof_stochastic_list_build + fof_link_stochastic_list: the potential edges written down once, every sample a
    stream over them.  Sample k = the oracle's sample (labels, potential and sampled edge counts bit-exact, log p
    to float64 summation order, score function to float32 order) = fof_link_stochastic(sample0 + k); records =
    2 x potential edges; a buffer that is too small reports the size it needs."""
    w = inputs.scaled(inputs.CONFIGS["cfg1"], 40)
    p = inputs.make_positions(w)
    p = np.ascontiguousarray(p[:len(p) - drop]) if drop else p
    b_link = w.b
    b_cand = float(np.float32(kappa * w.b))
    f = B.FoF(len(p), w.L, b_cand, w.N_min, path="cells")
    f.link(torch.from_numpy(p).cuda())
    small = torch.empty(B.fof_stochastic_list_bytes(f.h, 0), dtype=torch.uint8, device="cuda")
    records, filled = B.fof_stochastic_list_build(f.h, b_link, alpha, small, f.ws)
    o0 = oracle.stochastic(p, w.L, b_cand, b_link, alpha, 99, 3)
    assert not filled and records == 2 * o0["n_cand"]
    with pytest.raises(B.FofError) as e:      # a failed build leaves no valid list
        f.link_stochastic_list(small, 99, 3, 1)
    assert e.value.code == B.FOF_ERR_STATE
    slist, records2 = f.stochastic_list(b_link, alpha)
    assert records2 == records
    for want_grad in (True, False):
        labels, logp, grad = f.link_stochastic_list(slist, 99, 3, S, want_grad=want_grad)
        E_all, ncand, _ = f.link_stats()
        E_sum = 0
        for k in range(S):
            o = oracle.stochastic(p, w.L, b_cand, b_link, alpha, 99, 3 + k)
            assert ncand == o["n_cand"]
            E_sum += o["n_edge"]
            assert np.array_equal(labels[k].cpu().numpy(), o["labels"]), f"sample {k}: components differ"
            assert abs(float(logp[k].item()) - o["logp"]) <= 2e-6 * abs(o["logp"]) + 1e-6
            if want_grad:
                gk = grad[k].cpu().numpy().astype(np.float64)
                assert np.abs(gk - o["grad"]).max() <= 2e-5 * np.abs(o["grad"]).max()
        assert E_all == E_sum and (want_grad or grad is None)
    l1, lp1, g1 = f.link_stochastic(b_link, alpha, 99, 3)      # the list survives the calls that recompute
    la, lpa, ga = f.link_stochastic_list(slist, 99, 3, 1)
    assert torch.equal(l1, la[0])
    assert torch.allclose(g1, ga[0], rtol=0, atol=2e-5 * float(g1.abs().max()))
    f.link(torch.from_numpy(p).cuda())                         # ... but not a new link
    with pytest.raises(B.FofError) as e:
        f.link_stochastic_list(slist, 99, 3, 1)
    assert e.value.code == B.FOF_ERR_STATE
    f.close()


def test_stochastic_list_wraps(B):
    """n = 5 cells per axis: every candidate run wraps; brute-force oracle."""
    rng = np.random.default_rng(17)
    L, b = 8.0, 1.0
    p = (rng.random((3000, 3)) * L).astype(np.float32)
    f = B.FoF(len(p), L, 1.5, 5, path="cells")
    f.link(torch.from_numpy(p).cuda())
    slist, records = f.stochastic_list(b, 3.0)
    labels, logp, grad = f.link_stochastic_list(slist, 1, 0, 2)
    for k in range(2):
        o = oracle.stochastic(p, L, 1.5, b, 3.0, 1, k, brute=True)
        assert records == 2 * o["n_cand"]
        assert np.array_equal(labels[k].cpu().numpy(), o["labels"])
        assert abs(float(logp[k].item()) - o["logp"]) <= 2e-6 * abs(o["logp"])
        assert np.abs(grad[k].cpu().numpy() - o["grad"]).max() <= 2e-5 * np.abs(o["grad"]).max()
    f.close()


def test_groups_recounts_after_the_labels_buffer_was_reused(B):
    """fof_groups re-uses the sizes fof_link counted only for the labels fof_link wrote: once a stochastic sample has
    been written into the same buffer, the groups are those of the sample (counted afresh)."""
    w = inputs.scaled(inputs.CONFIGS["cfg1"], 32)
    p = inputs.make_positions(w)
    f = B.FoF(len(p), w.L, w.b, w.N_min, path="cells")
    dpos = torch.from_numpy(p).cuda()
    labels = f.link(dpos)
    logp = torch.zeros(1, dtype=torch.float64, device="cuda")
    B.fof_link_stochastic(f.h, w.b, 0.5, 11, 0, labels, logp, None, f.ws)      # overwrites `labels`
    g = f.groups(dpos, labels)
    lab = labels.cpu().numpy()
    og = oracle.groups(p, lab, w.L, w.N_min)
    det, _ = oracle.labels_cells(p, w.L, w.b)
    assert not np.array_equal(lab, det), "alpha = 0.5 should drop edges"
    assert g["K"] == og["K"] and np.array_equal(g["group_size"].cpu().numpy(), og["group_size"])
    f.close()


def test_stochastic_link_wraps_and_needs_a_link_first(B):
    rng = np.random.default_rng(17)
    L, b = 8.0, 1.0
    p = (rng.random((3000, 3)) * L).astype(np.float32)          # n = 5 cells per axis at b_cand = 1.5: every pair wraps
    f = B.FoF(len(p), L, 1.5, 5, path="cells")
    with pytest.raises(B.FofError) as e:
        f.link_stochastic(b, 3.0, 1, 0)
    assert e.value.code == B.FOF_ERR_STATE
    f.link(torch.from_numpy(p).cuda())
    o = oracle.stochastic(p, L, 1.5, b, 3.0, 1, 0, brute=True)
    labels, logp, grad = f.link_stochastic(b, 3.0, 1, 0)
    assert np.array_equal(labels.cpu().numpy(), o["labels"])
    assert abs(float(logp.item()) - o["logp"]) <= 2e-6 * abs(o["logp"])
    assert np.abs(grad.cpu().numpy() - o["grad"]).max() <= 2e-5 * np.abs(o["grad"]).max()
    f.close()


# --------------------------------------------------------------------------- NEXT-4: 6-D sub-halo pass
@pytest.mark.parametrize("sv_scale", [120.0, 1e15])
def test_subgroups_against_oracle(B, sv_scale):
    """fof_subgroups (section 2.1.1 Eq. 3): sub-halo labels bit-exact with the oracle (the same float32
    predicate on both sides), on halos that cross the box faces; sv -> infinity gives back the halos."""
    w = inputs.scaled(inputs.CONFIGS["cfg1"], 48)
    p = inputs.make_positions(w)
    rng = np.random.default_rng(19)
    v = (rng.standard_normal((len(p), 3)) * 50.0).astype(np.float32)
    lab, _ = oracle.labels_cells(p, w.L, w.b)
    og = oracle.groups(p, lab, w.L, w.N_min)
    pgo = og["particle_group"]
    v[(rng.random(len(p)) < 0.5) & (pgo >= 0)] += np.float32(400.0)      # a bulk flow through every halo
    ell = float(np.float32(1.3 * w.b))
    osub, _ = oracle.subgroups(p, v, pgo, w.L, 1.0, sv_scale ** 2, ell)

    f = B.FoF(len(p), w.L, w.b, w.N_min)
    dpos, dvel = torch.from_numpy(p).cuda(), torch.from_numpy(v).cuda()
    labels = f.link(dpos)
    g = f.groups(dpos, labels, particle_group=True)
    assert g["K"] == og["K"]
    sub = f.subgroups(dpos, dvel, g, 1.0, sv_scale ** 2, ell).cpu().numpy()
    assert np.array_equal(sub, osub), "sub-halo labels differ"
    if sv_scale > 1e10:
        assert np.array_equal(sub[pgo >= 0], lab[pgo >= 0])
    else:
        assert len(np.unique(sub[pgo >= 0])) > og["K"]
    # the link state was overwritten: a stochastic sample must ask for a new fof_link
    with pytest.raises(B.FofError) as e:
        f.link_stochastic(w.b, 1.0, 1, 0)
    assert e.value.code == B.FOF_ERR_STATE
    f.close()


def test_subgroups_large_halo_and_no_halo(B):
    rng = np.random.default_rng(23)
    L, b = 50.0, 1.0
    clump = rng.standard_normal((3000, 3)) * 1.2 + 25.0          # one halo of ~3000 members: 94 tiles
    p = np.concatenate([rng.random((2000, 3)) * L, clump]).astype(np.float32) % np.float32(L)
    v = (rng.standard_normal((len(p), 3)) * 30.0).astype(np.float32)
    v[2000:3500] += np.float32(200.0)
    lab, _ = oracle.labels_cells(p, L, b)
    og = oracle.groups(p, lab, L, 20)
    osub, _ = oracle.subgroups(p, v, og["particle_group"], L, 1.0, 60.0 ** 2, 0.9)
    f = B.FoF(len(p), L, b, 20)
    dpos, dvel = torch.from_numpy(p).cuda(), torch.from_numpy(v).cuda()
    g = f.groups(dpos, f.link(dpos), particle_group=True)
    assert g["group_size"].max().item() > 2000
    assert np.array_equal(f.subgroups(dpos, dvel, g, 1.0, 60.0 ** 2, 0.9).cpu().numpy(), osub)
    f.close()
    q = (rng.random((4000, 3)) * 100.0).astype(np.float32)        # no halo at all
    f = B.FoF(len(q), 100.0, 0.5, 20)
    dq = torch.from_numpy(q).cuda()
    g = f.groups(dq, f.link(dq), particle_group=True)
    assert g["K"] == 0
    sub = f.subgroups(dq, torch.zeros_like(dq), g, 1.0, 1.0, 1.0).cpu().numpy()
    assert np.array_equal(sub, np.arange(len(q), dtype=np.int32))
    f.close()


def test_subgroups_many_wide_halos_and_many_halos(B):
    """Several halos above the one-warp limit (their tile rows are dealt to the whole grid as work items found
    by a search of the item prefix), next to small ones, two of them across box faces; then more halos
    than one scan chunk (8192) so that the offsets come from two launches."""
    rng = np.random.default_rng(31)
    L, b = 60.0, 1.0
    centres = np.array([[0.2, 30, 30], [30, 59.9, 10], [15, 15, 15], [45, 20, 50], [50, 50, 0.1], [10, 40, 40]])
    sizes = [300, 700, 1500, 260, 257, 540]
    parts = [rng.standard_normal((m, 3)) * 0.9 + c for m, c in zip(sizes, centres)]
    small = [rng.standard_normal((int(m), 3)) * 0.35 + rng.random(3) * L for m in rng.integers(20, 200, 60)]
    p = (np.concatenate(parts + small + [rng.random((3000, 3)) * L]) % L).astype(np.float32)
    p = np.minimum(p, np.nextafter(np.float32(L), np.float32(0)))
    p = p[rng.permutation(len(p))]
    v = (rng.standard_normal((len(p), 3)) * 40.0).astype(np.float32)
    v[rng.random(len(p)) < 0.4] += np.float32(250.0)
    lab, _ = oracle.labels_cells(p, L, b)
    og = oracle.groups(p, lab, L, 20)
    assert (og["group_size"] > 256).sum() >= 5
    osub, _ = oracle.subgroups(p, v, og["particle_group"], L, 1.0, 70.0 ** 2, 0.8)
    f = B.FoF(len(p), L, b, 20)
    dpos, dvel = torch.from_numpy(p).cuda(), torch.from_numpy(v).cuda()
    g = f.groups(dpos, f.link(dpos), particle_group=True)
    sub = f.subgroups(dpos, dvel, g, 1.0, 70.0 ** 2, 0.8).cpu().numpy()
    assert np.array_equal(sub, osub)
    assert len(np.unique(sub[og["particle_group"] >= 0])) > og["K"]
    f.close()

    # 9000 pairs-of-clumps halos of 3 members each, N_min = 3: K > 8192
    K = 9000
    n = 24
    ij = np.stack(np.meshgrid(np.arange(n), np.arange(n), np.arange(n), indexing="ij"), -1).reshape(-1, 3)[:K]
    c = (ij + 0.5) * 4.0
    L2 = n * 4.0
    q = (c[:, None, :] + np.array([[0, 0, 0], [0.6, 0, 0], [0, 0.6, 0]])[None]).reshape(-1, 3).astype(np.float32)
    q = q[rng.permutation(len(q))]
    vq = (rng.standard_normal((len(q), 3)) * 30.0).astype(np.float32)
    lab, _ = oracle.labels_cells(q, L2, 1.0)
    og = oracle.groups(q, lab, L2, 3)
    assert og["K"] == K
    osub, _ = oracle.subgroups(q, vq, og["particle_group"], L2, 1.0, 40.0 ** 2, 0.9)
    f = B.FoF(len(q), L2, 1.0, 3)
    dq, dv = torch.from_numpy(q).cuda(), torch.from_numpy(vq).cuda()
    g = f.groups(dq, f.link(dq), particle_group=True)
    assert g["K"] == K
    assert np.array_equal(f.subgroups(dq, dv, g, 1.0, 40.0 ** 2, 0.9).cpu().numpy(), osub)
    f.close()


# --------------------------------------------------------------------------- NEXT-2: slab-decomposed FoF
@pytest.mark.parametrize("world", [2, 3, 4])
def test_slab_fof_equals_monolithic(B, world):
    """slabs + ghost layer + label-equivalence merge give exactly the monolithic labels
    (minimum global particle id).  All ranks are played in turn on this one GPU; the exchange is emulated."""
    from paper_2510_26851_b200 import slab

    w = inputs.scaled(inputs.CONFIGS["cfg1"], 48)
    p = inputs.make_positions(w)
    rng = np.random.default_rng(5)
    # a chain of particles 0.8 b apart along z through the whole box: one group that crosses every face
    nz = int(w.L / (0.8 * w.b))
    chain = np.stack([np.full(nz, 0.37 * w.L), np.full(nz, 0.61 * w.L), (np.arange(nz) + 0.5) * (w.L / nz)], 1)
    p = np.concatenate([p, chain.astype(np.float32)])
    p = p[rng.permutation(len(p))]
    N = len(p)
    f = B.FoF(N, w.L, w.b, w.N_min)
    mono = f.link(torch.from_numpy(p).cuda()).cpu().numpy()
    f.close()
    assert np.array_equal(mono, oracle.labels_cells(p, w.L, w.b)[0]), "monolithic labels differ from the oracle"
    own = slab.split_into_slabs(p, w.L, world)
    assert sum(len(o) for o in own) == N
    parts = [(torch.from_numpy(p[o]).cuda(), torch.from_numpy(o.astype(np.int32)).cuda()) for o in own]
    out = slab.slab_fof_emulated(parts, w.L, w.b, N)
    crossing = 0
    for o, lab in zip(own, out):
        assert np.array_equal(lab.cpu().numpy(), mono[o]), "slab labels differ from the monolithic run"
        crossing += int((~np.isin(mono[o], o)).sum())
    assert crossing > nz // 2          # many particles whose canonical particle lives on another rank


@pytest.mark.parametrize("world,weighted", [(2, False), (3, True), (4, True)])
def test_slab_groups_against_oracle(B, world, weighted):
    """Cross-rank group construction ("identical to a monolithic run" PAPER.md:180): the union of
    the per-rank catalogues of a 2 / 3 / 4-slab run (all ranks played in turn on this GPU) is the oracle's
    catalogue of the whole box: labels and sizes exact, masses 1e-5 relative, centres of mass 1e-5 L.  The set
    holds groups inside one slab, groups across a slab face, across the box face in z, and a chain through every
    slab whose canonical particle lives on one rank only."""
    from paper_2510_26851_b200 import slab

    w = inputs.scaled(inputs.CONFIGS["cfg1"], 48)
    p = inputs.make_positions(w)
    rng = np.random.default_rng(7 + world)
    nz = int(w.L / (0.8 * w.b))
    chain = np.stack([np.full(nz, 0.37 * w.L), np.full(nz, 0.61 * w.L), (np.arange(nz) + 0.5) * (w.L / nz)], 1)
    p = np.concatenate([p, chain.astype(np.float32)])
    p = p[rng.permutation(len(p))]
    N = len(p)
    mass = rng.uniform(0.5, 1.5, N).astype(np.float32) if weighted else None
    N_min = 5
    lab, _ = oracle.labels_cells(p, w.L, w.b)
    og = oracle.groups(p, lab, w.L, N_min, mass=mass)
    own = slab.split_into_slabs(p, w.L, world)
    parts = [(torch.from_numpy(p[o]).cuda(), torch.from_numpy(o.astype(np.int32)).cuda()) for o in own]
    masses = None if mass is None else [torch.from_numpy(mass[o]).cuda() for o in own]
    labels, cats = slab.slab_fof_emulated(parts, w.L, w.b, N, N_min=N_min, masses=masses)
    for o, l in zip(own, labels):
        assert np.array_equal(l.cpu().numpy(), lab[o])
    glab = np.concatenate([c["group_label"].cpu().numpy() for c in cats])
    order = np.argsort(glab)
    assert sum(c["K"] for c in cats) == og["K"]
    assert np.array_equal(glab[order], og["group_label"]), "the ranks' catalogues do not add up to the oracle's"
    for c, o in zip(cats, own):
        assert np.isin(c["group_label"].cpu().numpy(), o).all(), "a rank lists a group whose canonical particle it does not own"
    size = np.concatenate([c["group_size"].cpu().numpy() for c in cats])[order]
    gm = np.concatenate([c["group_mass"].cpu().numpy() for c in cats])[order]
    com = np.concatenate([c["group_com"].cpu().numpy() for c in cats])[order]
    assert np.array_equal(size, og["group_size"])
    assert np.all(np.abs(gm - og["group_mass"]) <= 1e-5 * og["group_mass"])
    d = np.abs(com.astype(np.float64) - og["group_com"])
    d = np.minimum(d, float(np.float32(w.L)) - d)
    assert d.max() <= 1e-5 * w.L, f"centre of mass off by {d.max()}"
    spanning = sum(int((~np.isin(lab[o], o)).any()) for o in own)
    assert og["group_size"].max() >= nz and spanning >= world - 1   # the chain is one group over all slabs


@pytest.mark.parametrize("grid", [3, 4, 5, 6, 7])
def test_tiny_grids_wrap_everywhere(B, grid):
    """n = 3 .. 5 cells per axis: every stencil wraps and the minimum-image selects are live in both roles
    of the link kernel; n = 6, 7: the first grids where interior warps take the wrap-free variant.  Dense
    clumps on the box corner and faces plus a sparse background."""
    rng = np.random.default_rng(100 + grid)
    L, b = 10.0, 1.0
    corner = rng.standard_normal((400, 3)) * 0.5                      # straddles all three faces at 0 / L
    face = rng.standard_normal((300, 3)) * 0.4 + np.array([5.0, 0.0, 5.0])
    bg = rng.random((1500, 3)) * L
    p = (np.concatenate([corner, face, bg]) % L).astype(np.float32)
    p[p >= np.float32(L)] = 0.0
    p = p[rng.permutation(len(p))]
    got, lab, og = check_against_oracle(B, p, L, b, 5, grid=grid, brute=True,
                                        mass=rng.uniform(0.5, 1.5, len(p)).astype(np.float32))
    assert got["grid"][0] == grid and og["group_size"].max() > 300


@pytest.mark.parametrize("grid", [3, 5, 8])
def test_heavy_cells_across_the_wrap(B, grid):
    """Cells of several hundred particles on both sides of the box faces: their tiles are listed as eight
    work items each (the candidate stream of a heavy cell is shared out, kernels_link.cu), with wrapping
    neighbours (n = 3, 5) and with the wrap-free variant next to wrapping ones (n = 8)."""
    rng = np.random.default_rng(200 + grid)
    L, b = 10.0, 1.0
    corner = rng.standard_normal((2400, 3)) * 0.45                    # ~300 per cell in the eight corner cells
    edge = rng.standard_normal((900, 3)) * 0.35 + np.array([0.0, 5.0, 0.0])
    inner = rng.standard_normal((700, 3)) * 0.3 + np.array([5.2, 5.1, 4.9])
    bg = rng.random((1000, 3)) * L
    p = (np.concatenate([corner, edge, inner, bg]) % L).astype(np.float32)
    p[p >= np.float32(L)] = 0.0
    p = p[rng.permutation(len(p))]
    got, lab, og = check_against_oracle(B, p, L, b, 5, grid=grid, brute=True,
                                        mass=rng.uniform(0.5, 1.5, len(p)).astype(np.float32))
    assert got["grid"][0] == grid and og["group_size"].max() > 2000

