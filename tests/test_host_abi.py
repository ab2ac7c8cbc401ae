"""CPU-only checks of the boundary: the C-ABI library loads and exports every symbol that
include/fof.h declares, the host-only calls behave as the header says (no compute call is made:
there is no GPU here), and the multi-rank bookkeeping of bench.py works under gloo, world size 2."""
from __future__ import annotations

import ctypes
import json
import os
import re
import subprocess
import sys

import numpy as np
import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def B():
    from paper_2510_26851_b200 import binding, build

    build.build()
    binding.lib()
    return binding


def declared_symbols():
    text = open(os.path.join(ROOT, "include", "fof.h")).read()
    text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)
    return sorted(set(re.findall(r"\b(fof_[a-z_]+)\s*\(", text)))


def test_library_exports_every_declared_symbol(B):
    names = declared_symbols()
    assert len(names) >= 18 and "fof_link" in names and "fof_groups" in names and "fof_create" in names
    raw = ctypes.CDLL(B.LIB_PATH)
    for n in names:
        assert hasattr(raw, n), f"{n} is declared in include/fof.h but not exported"


def test_plan_and_argument_errors(B):
    # Eq. 1: b = b_frac L / N^(1/3), evaluated in double, rounded once
    assert B.fof_linking_length(0.2, 1000.0, 256 ** 3) == float(np.float32(0.2 * 1000.0 / 256))
    h = B.fof_create(256 ** 3, 1000.0, 0.78125, 20)
    n, cells, n_max = B.fof_get_grid(h)
    assert n == 256 and cells == 256 ** 3 and n_max == 1024   # floor(1280 / 1.001) = 1278, capped at 1024
    ws = B.fof_workspace_bytes(h)
    assert 256 ** 3 * 50 < ws < 256 ** 3 * 120
    B.fof_set_grid(h, 128)
    assert B.fof_get_grid(h)[0] == 128 and B.fof_workspace_bytes(h) < ws
    with pytest.raises(B.FofError) as e:
        B.fof_set_grid(h, 2000)
    assert e.value.code == B.FOF_ERR_INVALID_ARG
    B.fof_destroy(h)
    for bad in [(-1, 1.0, 0.1, 20), (10, 0.0, 0.1, 20), (10, 1.0, -0.1, 20), (10, 1.0, 0.1, 0), (2 ** 31, 1.0, 0.1, 20)]:
        with pytest.raises(B.FofError) as e:
            B.fof_create(*bad)
        assert e.value.code == B.FOF_ERR_INVALID_ARG
    with pytest.raises(B.FofError) as e:      # fewer than 3 cells of side >= b per axis
        B.fof_create(100, 1.0, 0.4, 20)
    assert e.value.code == B.FOF_ERR_UNSUPPORTED
    h = B.fof_create(0, 1.0, 0.1, 20)          # N = 0 is a valid plan
    assert B.fof_workspace_bytes(h) > 0
    B.fof_destroy(h)
    assert B.lib().fof_error_string(B.FOF_ERR_CAPACITY).decode() == "more groups than capacity"
    assert B.lib().fof_error_string(12345).decode() == "unknown error"


def test_stochastic_batch_argument_and_state_errors(B):
    """fof_link_stochastic_batch rejects bad arguments and a missing fof_link before it touches any memory."""
    import ctypes

    L = B.lib()
    h = B.fof_create(1000, 10.0, 1.0, 5)
    assert L.fof_stochastic_scratch_bytes(h, 3) == 3 * 1001 * 4
    assert L.fof_stochastic_scratch_bytes(h, 0) == 0 and L.fof_stochastic_scratch_bytes(None, 3) == 0
    raw = np.zeros(4096, dtype=np.uint8)
    addr = (raw.ctypes.data + 255) & ~255            # a 256-B aligned host address: never dereferenced here
    p = ctypes.c_void_p(addr)
    call = lambda b_link, alpha, S, ws=p: L.fof_link_stochastic_batch(h, ctypes.c_float(b_link), ctypes.c_float(alpha), 1, 0,
                                                                      S, p, p, None, p, ws, None)
    assert call(1.0, 2.0, 0) == B.FOF_ERR_INVALID_ARG          # no samples
    assert call(1.0, 2.0, 2000) == B.FOF_ERR_INVALID_ARG       # too many
    assert call(1.5, 2.0, 2) == B.FOF_ERR_INVALID_ARG          # b_link above the plan's candidate radius
    assert call(1.0, float("nan"), 2) == B.FOF_ERR_INVALID_ARG
    assert call(1.0, 2.0, 2, ctypes.c_void_p(addr + 4)) == B.FOF_ERR_INVALID_ARG   # workspace not 256-B aligned
    assert call(1.0, 2.0, 2) == B.FOF_ERR_STATE                # no fof_link on this (handle, workspace) yet
    B.fof_destroy(h)


def test_stochastic_list_argument_and_state_errors(B):
    """The potential-edge list calls reject bad arguments and a missing fof_link / build before touching memory."""
    import ctypes

    L = B.lib()
    h = B.fof_create(1000, 10.0, 1.0, 5)
    fixed = L.fof_stochastic_list_bytes(h, 0)
    assert fixed >= 256 + 1001 * 4 + 1000 * 4 and fixed % 256 == 0
    assert L.fof_stochastic_list_bytes(h, 10) == fixed + 320 and L.fof_stochastic_list_bytes(None, 10) == 0
    raw = np.zeros(4096, dtype=np.uint8)
    p = ctypes.c_void_p((raw.ctypes.data + 255) & ~255)        # 256-B aligned host address: never dereferenced here
    odd = ctypes.c_void_p(p.value + 4)
    R = ctypes.c_uint64()
    build = lambda b_link, alpha, lst=p, nbytes=fixed, ws=p: L.fof_stochastic_list_build(
        h, ctypes.c_float(b_link), ctypes.c_float(alpha), lst, nbytes, ctypes.byref(R), ws, None)
    assert build(1.5, 2.0) == B.FOF_ERR_INVALID_ARG            # b_link above the plan's candidate radius
    assert build(1.0, float("inf")) == B.FOF_ERR_INVALID_ARG
    assert build(1.0, 2.0, lst=odd) == B.FOF_ERR_INVALID_ARG   # list not 256-B aligned
    assert build(1.0, 2.0, ws=odd) == B.FOF_ERR_INVALID_ARG
    assert build(1.0, 2.0, nbytes=fixed - 1) == B.FOF_ERR_INVALID_ARG   # not even room for the offsets
    assert build(1.0, 2.0) == B.FOF_ERR_STATE                  # no fof_link on this (handle, workspace) yet
    run = lambda S, lst=p: L.fof_link_stochastic_list(h, lst, 1, 0, S, p, p, None, p, p, None)
    assert run(0) == B.FOF_ERR_INVALID_ARG and run(2000) == B.FOF_ERR_INVALID_ARG
    assert run(2, lst=None) == B.FOF_ERR_INVALID_ARG
    assert run(2) == B.FOF_ERR_STATE                           # no list was built
    B.fof_destroy(h)


def test_grid_choice_keeps_cell_side_above_b(B):
    """H0: cell side L/n >= 1.001 b for every plan (R3), n >= 3."""
    rng = np.random.default_rng(1)
    for _ in range(200):
        L = float(np.float32(10 ** rng.uniform(-2, 4)))
        b = float(np.float32(L / rng.uniform(3.2, 5000)))
        N = int(10 ** rng.uniform(0, 9))
        h = B.fof_create(N, L, b, 20)
        n, cells, n_max = B.fof_get_grid(h)
        assert 3 <= n <= n_max <= 1024 and cells == n ** 3
        assert L / n_max >= b * 1.001 * (1 - 1e-6)
        B.fof_destroy(h)


def _gloo_worker(rank, world, port, out):
    import torch.distributed as dist

    os.environ.update(RANK=str(rank), LOCAL_RANK=str(rank), WORLD_SIZE=str(world), MASTER_ADDR="127.0.0.1",
                      MASTER_PORT=str(port))
    sys.path.insert(0, ROOT)
    import bench

    dist.init_process_group("gloo", rank=rank, world_size=world)
    assert bench.dist_env() == (rank, rank, world)
    w = bench.workload_for_rank("cfg0", rank)
    ms = bench.max_over_ranks_ms(10.0 + 5.0 * rank, world, "cpu")   # rank 1 is the slow one
    out.put((rank, w.seed, w.N, ms, bench.whole_job_value(world, w.N, ms)))
    dist.barrier()
    dist.destroy_process_group()


def test_replica_bookkeeping_under_gloo_world_2():
    import torch.multiprocessing as mp

    ctx = mp.get_context("spawn")
    out = ctx.Queue()
    port = 29500 + os.getpid() % 2000
    procs = [ctx.Process(target=_gloo_worker, args=(r, 2, port, out)) for r in range(2)]
    for p in procs:
        p.start()
    rows = sorted(out.get(timeout=120) for _ in procs)
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    (r0, s0, n0, ms0, v0), (r1, s1, n1, ms1, v1) = rows
    assert s0 != s1 and n0 == n1 == 32 ** 3            # independent replicas of the same workload
    assert ms0 == ms1 == 15.0                           # max over ranks
    assert v0 == v1 == 2 * 32 ** 3 / 15.0e-3            # whole-job aggregate


def test_reference_arm_other_ranks_exit_silently():
    env = dict(os.environ, RANK="1", LOCAL_RANK="1", WORLD_SIZE="2")
    r = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--gpus", "2",
                        "--steps", "1", "--warmup", "0"], env=env, capture_output=True, text=True, timeout=120)
    assert r.returncode == 0 and r.stdout.strip() == ""


def test_reference_arm_prints_the_contract_line():
    r = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--steps", "1",
                        "--warmup", "0", "--workload", "cfg0"], capture_output=True, text=True, timeout=300)
    assert r.returncode == 0, r.stderr
    line = json.loads(r.stdout.strip().splitlines()[-1])
    assert line["impl"] == "reference" and line["metric"] == "fof_linked_particles_per_s"
    assert line["cpu_baseline"]["kind"] == "oracle" and line["e2e"]["h2d_bytes_per_step"] == 0
    assert line["value"] > 0 and line["config"]["workload"] == "cfg0"


def _ring_worker(rank, world, port, out):
    import torch
    import torch.distributed as dist

    os.environ.update(RANK=str(rank), LOCAL_RANK=str(rank), WORLD_SIZE=str(world), MASTER_ADDR="127.0.0.1",
                      MASTER_PORT=str(port))
    sys.path.insert(0, ROOT)
    from paper_2510_26851_b200.slab import RingExchange

    dist.init_process_group("gloo", rank=rank, world_size=world)
    ex = RingExchange()
    # rank r lends r + 1 rows (rank 0: also tests the empty case when world == 3 via rank 2 -> 0 rows)
    rows = 0 if (world == 3 and rank == 2) else rank + 1
    t = torch.full((rows, 3), float(rank)) + torch.arange(3.0)
    got = ex.send_down_recv_up(t)                       # rows lent by rank + 1
    ids = ex.send_down_recv_up(torch.arange(rows, dtype=torch.int32) + 100 * rank)
    pairs = torch.tensor([[rank, 10 + rank]] * rank, dtype=torch.int32).reshape(rank, 2)
    allp = ex.all_gather_rows(pairs)
    out.put((rank, got.tolist(), ids.tolist(), allp.tolist()))
    dist.barrier()
    dist.destroy_process_group()


@pytest.mark.parametrize("world", [2, 3])
def test_slab_ring_exchange_under_gloo(world):
    """The plumbing of the slab-decomposed FoF (NEXT-2): variable-length ring send/recv (who lends to whom,
    empty messages) and the all-gather of the equivalence pairs, on CPU tensors over gloo."""
    import torch.multiprocessing as mp

    ctx = mp.get_context("spawn")
    out = ctx.Queue()
    port = 31500 + (os.getpid() + world) % 2000
    procs = [ctx.Process(target=_ring_worker, args=(r, world, port, out)) for r in range(world)]
    for p in procs:
        p.start()
    rows = sorted(out.get(timeout=120) for _ in procs)
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    for rank, got, ids, allp in rows:
        up = (rank + 1) % world
        n_up = 0 if (world == 3 and up == 2) else up + 1
        assert got == [[float(up), float(up) + 1, float(up) + 2]] * n_up      # what rank + 1 lent
        assert ids == [100 * up + k for k in range(n_up)]
        assert allp == [[r, 10 + r] for r in range(world) for _ in range(r)]    # rank-major concatenation
