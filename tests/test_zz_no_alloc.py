"""fof_group_sigma_static: the halo decoration with the library's static device scratch instead of a caller
workspace (for callers that cannot allocate: include/fof.h).  Checked against the existing path, fof_group_sigma,
within the tolerance of test_sigma_and_backward_against_oracle, on two calls in a row that share the scratch array
(the second on other data with fewer groups: stale sums of the first call would show), and against the oracle.
Collected last on purpose (the suite runs with pytest -x).
"""
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


def _case(B, n_side, weighted, seed_shift):
    import dataclasses

    w = inputs.scaled(inputs.CONFIGS["cfg1"], n_side)
    w = dataclasses.replace(w, seed=w.seed + seed_shift)
    p = inputs.make_positions(w)
    m = inputs.make_masses(w) if weighted else None
    f = B.FoF(len(p), w.L, w.b, w.N_min)
    dpos = torch.from_numpy(p).cuda()
    dm = None if m is None else torch.from_numpy(m).cuda()
    g = f.groups(dpos, f.link(dpos), mass=dm, particle_group=True)
    return w, p, m, f, dpos, dm, g


def test_static_scratch_sigma_equals_the_workspace_path_twice_in_a_row(B):
    first = _case(B, 48, True, 0)
    second = _case(B, 32, False, 77)      # fewer groups, unit masses: must not see the first call's sums
    assert first[6]["K"] > second[6]["K"] > 0
    for w, p, m, f, dpos, dm, g in (first, second):
        K = g["K"]
        assert K <= B.FOF_SIGMA_STATIC_MAX_GROUPS
        want = f.group_sigma(dpos, g, mass=dm)                       # existing path: scratch in the workspace
        got = torch.full((K,), -1.0, dtype=torch.float32, device="cuda")
        B.fof_group_sigma_static(f.h, dpos, dm, g["particle_group"], g["group_mass"], g["group_com"], K, got)
        torch.cuda.synchronize()
        a, b = got.cpu().numpy().astype(np.float64), want.cpu().numpy().astype(np.float64)
        assert np.all(a > 0)
        assert np.all(np.abs(a - b) <= 2e-6 * b + 1e-7 * w.L)       # float64 atomics in another order
        lab, _ = oracle.labels_cells(p, w.L, w.b)
        og = oracle.groups(p, lab, w.L, w.N_min, mass=m)
        osig = oracle.group_sigma(p, og["particle_group"], w.L, og["group_com"], mass=m)
        assert og["K"] == K and np.all(np.abs(a - osig) <= 2e-6 * osig + 1e-7 * w.L)
    # the same call again on the first data (the array now holds the second call's sums)
    w, p, m, f, dpos, dm, g = first
    again = torch.empty(g["K"], dtype=torch.float32, device="cuda")
    B.fof_group_sigma_static(f.h, dpos, dm, g["particle_group"], g["group_mass"], g["group_com"], g["K"], again)
    want = f.group_sigma(dpos, g, mass=dm).cpu().numpy().astype(np.float64)
    assert np.all(np.abs(again.cpu().numpy().astype(np.float64) - want) <= 2e-6 * want + 1e-7 * w.L)
    for c in (first, second):
        c[3].close()


def test_static_scratch_rejects_more_groups_than_it_holds(B):
    """K beyond FOF_SIGMA_STATIC_MAX_GROUPS: FOF_ERR_CAPACITY before anything is launched or dereferenced."""
    N = B.FOF_SIGMA_STATIC_MAX_GROUPS + 10
    h = B.fof_create(N, 100.0, 0.1, 1)                              # N_min = 1: up to N groups
    x = torch.zeros(16, dtype=torch.float32, device="cuda")         # stand-ins: never read
    with pytest.raises(B.FofError) as e:
        B.fof_group_sigma_static(h, x, None, x, x, x, B.FOF_SIGMA_STATIC_MAX_GROUPS + 1, x)
    assert e.value.code == B.FOF_ERR_CAPACITY
    with pytest.raises(B.FofError) as e:
        B.fof_group_sigma_static(h, x, None, x, x, x, N + 1, x)     # more groups than particles: as fof_group_sigma
    assert e.value.code == B.FOF_ERR_INVALID_ARG
    B.fof_group_sigma_static(h, x, None, x, x, x, 0, x)             # K = 0: nothing to do
    torch.cuda.synchronize()
    B.fof_destroy(h)
