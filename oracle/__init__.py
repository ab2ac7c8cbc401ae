"""ctypes wrapper around oracle/fof_oracle.c — the CPU oracle.

TEST INFRASTRUCTURE, NOT PRODUCT: only tests/, __graft_entry__.smoke() and bench.py's
cpu_baseline / --impl reference legs may import this package.  It imports nothing from
paper_2510_26851_b200 and shares no code with the CUDA path.

Every function cites the passage of the paper it follows in oracle/fof_oracle.c.
"""
from __future__ import annotations

import ctypes
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "fof_oracle.c")
_SRC2 = os.path.join(_HERE, "fof_oracle_stochastic.c")  # NEXT-3: stochastic-edge FoF
_SRC3 = os.path.join(_HERE, "fof_oracle_subhalo.c")     # NEXT-4: six-dimensional sub-halo pass
_LIB = os.path.join(_HERE, "libfof_oracle.so")
# -ffp-contract=off: the float32 link predicate must not be contracted into FMAs.
CFLAGS = ["-O2", "-std=c99", "-ffp-contract=off", "-fno-fast-math", "-fopenmp", "-shared", "-fPIC"]

_lib = None


def build(force: bool = False) -> str:
    """Compile the oracle with gcc (building the checker is not using it)."""
    newest = max(os.path.getmtime(_SRC), os.path.getmtime(_SRC2), os.path.getmtime(_SRC3))
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < newest:
        tmp = _LIB + f".tmp{os.getpid()}"
        subprocess.check_call(["gcc", *CFLAGS, "-o", tmp, _SRC, _SRC2, _SRC3, "-lm"])
        os.replace(tmp, _LIB)
    return _LIB


def _load():
    global _lib
    if _lib is None:
        lib = ctypes.CDLL(build())
        f32p = ctypes.POINTER(ctypes.c_float)
        i32p = ctypes.POINTER(ctypes.c_int32)
        f64p = ctypes.POINTER(ctypes.c_double)
        u64p = ctypes.POINTER(ctypes.c_uint64)
        lib.oracle_wrap1.restype = ctypes.c_float
        lib.oracle_wrap1.argtypes = [ctypes.c_float, ctypes.c_float]
        lib.oracle_wrap.restype = ctypes.c_int
        lib.oracle_wrap.argtypes = [f32p, ctypes.c_int64, ctypes.c_float, f32p]
        lib.oracle_link.restype = ctypes.c_int
        lib.oracle_link.argtypes = [f32p, f32p, ctypes.c_float, ctypes.c_float]
        for fn in (lib.oracle_labels_brute, lib.oracle_labels_cells):
            fn.restype = ctypes.c_int
            fn.argtypes = [f32p, ctypes.c_int64, ctypes.c_float, ctypes.c_float, i32p, u64p]
        lib.oracle_labels_cells_threads.restype = ctypes.c_int
        lib.oracle_labels_cells_threads.argtypes = [f32p, ctypes.c_int64, ctypes.c_float, ctypes.c_float, i32p, u64p,
                                                    ctypes.c_int32]
        lib.oracle_groups.restype = ctypes.c_int64
        lib.oracle_groups.argtypes = [f32p, f32p, i32p, ctypes.c_int64, ctypes.c_float, ctypes.c_int32,
                                      ctypes.c_int64, i32p, i32p, f64p, f64p, i32p]
        f64p_ = ctypes.POINTER(ctypes.c_double)
        lib.oracle_group_sigma.restype = ctypes.c_int
        lib.oracle_group_sigma.argtypes = [f32p, f32p, i32p, ctypes.c_int64, ctypes.c_float, ctypes.c_int64, f64p_,
                                           f64p_]
        lib.oracle_groups_backward.restype = ctypes.c_int
        lib.oracle_groups_backward.argtypes = [f32p, f32p, i32p, ctypes.c_int64, ctypes.c_float, ctypes.c_int64,
                                               f64p_, f64p_, f64p_, f64p_, f64p_, f64p_]
        f64q = ctypes.POINTER(ctypes.c_double)
        lib.oracle_subgroups.restype = ctypes.c_int
        lib.oracle_subgroups.argtypes = [f32p, f32p, i32p, ctypes.c_int64, ctypes.c_float, ctypes.c_float,
                                         ctypes.c_float, ctypes.c_float, i32p, u64p]
        lib.oracle_sigmoid_fixed.restype = ctypes.c_float
        lib.oracle_sigmoid_fixed.argtypes = [ctypes.c_float]
        lib.oracle_rng_u24.restype = ctypes.c_uint32
        lib.oracle_rng_u24.argtypes = [ctypes.c_uint64, ctypes.c_uint32, ctypes.c_uint32, ctypes.c_uint32]
        for fn in (lib.oracle_stochastic_brute, lib.oracle_stochastic_cells):
            fn.restype = ctypes.c_int
            fn.argtypes = [f32p, ctypes.c_int64, ctypes.c_float, ctypes.c_float, ctypes.c_float, ctypes.c_float,
                           ctypes.c_uint64, ctypes.c_uint32, i32p, f64q, f64q, u64p, u64p]
        lib.oracle_stochastic_edges.restype = ctypes.c_int64
        lib.oracle_stochastic_edges.argtypes = [f32p, ctypes.c_int64, ctypes.c_float, ctypes.c_float, ctypes.c_float,
                                                ctypes.c_float, ctypes.c_uint64, ctypes.c_uint32, ctypes.c_int64,
                                                i32p, i32p, f32p]
        lib.oracle_pref.restype = ctypes.c_int
        lib.oracle_pref.argtypes = [f32p, ctypes.c_int64, ctypes.c_float, ctypes.c_float, u64p]
        lib.oracle_linking_length.restype = ctypes.c_float
        lib.oracle_linking_length.argtypes = [ctypes.c_float, ctypes.c_float, ctypes.c_int64]
        _lib = lib
    return _lib


def _f(x) -> float:
    """round once to float32 (what the C side receives), as a Python float for ctypes."""
    return float(np.float32(x))


class OracleError(RuntimeError):
    pass


def _f32(a):
    a = np.ascontiguousarray(a, dtype=np.float32)
    return a, a.ctypes.data_as(ctypes.POINTER(ctypes.c_float))


def _pos(pos):
    pos = np.ascontiguousarray(pos, dtype=np.float32).reshape(-1, 3)
    return pos, pos.ctypes.data_as(ctypes.POINTER(ctypes.c_float))


def _check(rc):
    if rc < 0:
        raise OracleError({-1: "bad argument", -2: "non-finite position", -3: "out of memory"}.get(int(rc), str(rc)))
    return rc


def wrap1(x: float, L: float) -> float:
    return float(_load().oracle_wrap1(_f(x), _f(L)))


def wrap(pos, L: float) -> np.ndarray:
    pos, p = _pos(pos)
    out = np.empty_like(pos)
    _check(_load().oracle_wrap(p, pos.shape[0], _f(L), out.ctypes.data_as(ctypes.POINTER(ctypes.c_float))))
    return out


def link(wi, wj, L: float, b: float) -> bool:
    wi, pi = _f32(wi)
    wj, pj = _f32(wj)
    return bool(_load().oracle_link(pi, pj, _f(L), _f(b)))


def _labels(fn, pos, L, b):
    pos, p = _pos(pos)
    N = pos.shape[0]
    labels = np.empty(N, dtype=np.int32)
    E = ctypes.c_uint64(0)
    _check(fn(p, N, _f(L), _f(b), labels.ctypes.data_as(ctypes.POINTER(ctypes.c_int32)),
              ctypes.byref(E)))
    return labels, int(E.value)


def labels_brute(pos, L: float, b: float):
    """(labels int32 [N], E) by all-pairs + min-label sweeps. O(N^2): tiny inputs only."""
    return _labels(_load().oracle_labels_brute, pos, L, b)


def labels_cells(pos, L: float, b: float):
    """(labels int32 [N], E) by cell list + sequential union-find."""
    return _labels(_load().oracle_labels_cells, pos, L, b)


def labels_cells_threads(pos, L: float, b: float, threads: int):
    """(labels, E) like labels_cells, the pair search on `threads` host threads (serial union step): only for the
    all-cores CPU figure of bench.py; parity uses labels_cells."""
    pos, p = _pos(pos)
    N = pos.shape[0]
    labels = np.empty(N, dtype=np.int32)
    E = ctypes.c_uint64(0)
    fn = _load().oracle_labels_cells_threads
    _check(fn(p, N, _f(L), _f(b), labels.ctypes.data_as(ctypes.POINTER(ctypes.c_int32)), ctypes.byref(E), int(threads)))
    return labels, int(E.value)


def groups(pos, labels, L: float, N_min: int, mass=None):
    """dict(K, group_label, group_size, group_mass f64, group_com f64 [K,3], particle_group)."""
    pos, p = _pos(pos)
    N = pos.shape[0]
    labels = np.ascontiguousarray(labels, dtype=np.int32)
    cap = max(1, N // max(1, int(N_min)))
    gl = np.empty(cap, np.int32)
    gs = np.empty(cap, np.int32)
    gm = np.empty(cap, np.float64)
    gc = np.empty((cap, 3), np.float64)
    pg = np.empty(N, np.int32)
    mp = None
    if mass is not None:
        mass, mp = _f32(mass)
    i32p = ctypes.POINTER(ctypes.c_int32)
    f64p = ctypes.POINTER(ctypes.c_double)
    K = _check(_load().oracle_groups(p, mp, labels.ctypes.data_as(i32p), N, _f(L), int(N_min), cap,
                                     gl.ctypes.data_as(i32p), gs.ctypes.data_as(i32p), gm.ctypes.data_as(f64p),
                                     gc.ctypes.data_as(f64p), pg.ctypes.data_as(i32p)))
    K = int(K)
    return dict(K=K, group_label=gl[:K].copy(), group_size=gs[:K].copy(), group_mass=gm[:K].copy(),
                group_com=gc[:K].copy(), particle_group=pg)


def _f64(a):
    if a is None:
        return None, None
    a = np.ascontiguousarray(a, dtype=np.float64)
    return a, a.ctypes.data_as(ctypes.POINTER(ctypes.c_double))


def group_sigma(pos, particle_group, L: float, group_com, mass=None) -> np.ndarray:
    """sigma_g = sqrt(sum m |min-image(w_i - X_g)|^2 / M_g), float64 [K] (section 3.1.1, reading R23)."""
    pos, p = _pos(pos)
    pg = np.ascontiguousarray(particle_group, dtype=np.int32)
    gc, gcp = _f64(group_com)
    K = gc.shape[0]
    out = np.zeros(max(K, 1), np.float64)
    mp = None
    if mass is not None:
        mass, mp = _f32(mass)
    _check(_load().oracle_group_sigma(p, mp, pg.ctypes.data_as(ctypes.POINTER(ctypes.c_int32)), pos.shape[0], _f(L),
                                      K, gcp, out.ctypes.data_as(ctypes.POINTER(ctypes.c_double))))
    return out[:K]


def groups_backward(pos, particle_group, L: float, group_mass, group_com, grad_com, group_sigma=None,
                    grad_sigma=None, mass=None) -> np.ndarray:
    """Frozen-assignment backward (Eq. 4; Eq. 5 through sigma): float64 [N,3]."""
    pos, p = _pos(pos)
    N = pos.shape[0]
    pg = np.ascontiguousarray(particle_group, dtype=np.int32)
    gm, gmp = _f64(group_mass)
    gc, gcp = _f64(group_com)
    gs, gsp = _f64(group_sigma)
    dx, dxp = _f64(grad_com)
    ds, dsp = _f64(grad_sigma)
    out = np.zeros((max(N, 1), 3), np.float64)
    mp = None
    if mass is not None:
        mass, mp = _f32(mass)
    _check(_load().oracle_groups_backward(p, mp, pg.ctypes.data_as(ctypes.POINTER(ctypes.c_int32)), N, _f(L),
                                          gm.shape[0], gmp, gcp, gsp, dxp, dsp,
                                          out.ctypes.data_as(ctypes.POINTER(ctypes.c_double))))
    return out[:N]


def subgroups(pos, vel, particle_group, L: float, sigma_x: float, sigma_v: float, ell: float):
    """Six-dimensional FoF inside every kept halo (Eq. 3): (sub_labels int32 [N], E6)."""
    pos, p = _pos(pos)
    vel, v = _f32(vel)
    N = pos.shape[0]
    pg = np.ascontiguousarray(particle_group, dtype=np.int32)
    out = np.empty(max(N, 1), np.int32)
    E = ctypes.c_uint64(0)
    i32p = ctypes.POINTER(ctypes.c_int32)
    _check(_load().oracle_subgroups(p, v, pg.ctypes.data_as(i32p), N, _f(L), _f(sigma_x), _f(sigma_v), _f(ell),
                                    out.ctypes.data_as(i32p), ctypes.byref(E)))
    return out[:N], int(E.value)


def sigmoid_fixed(t: float) -> float:
    """The fixed float32 logistic of reading R26 (NEXT-3)."""
    return float(_load().oracle_sigmoid_fixed(_f(t)))


def rng_u24(seed: int, sample: int, lo: int, hi: int) -> int:
    """24 random bits of the counter-based generator of reading R27 (NEXT-3)."""
    return int(_load().oracle_rng_u24(int(seed), int(sample), int(lo), int(hi)))


def stochastic(pos, L: float, b_cand: float, b_link: float, alpha: float, seed: int, sample: int, brute=False,
               want_grad=True):
    """One Monte Carlo sample of stochastic-edge FoF (Eq. 8): dict(labels, logp, grad [N,3] f64,
    n_cand, n_edge)."""
    pos, p = _pos(pos)
    N = pos.shape[0]
    labels = np.empty(max(N, 1), np.int32)
    grad = np.zeros((max(N, 1), 3), np.float64) if want_grad else None
    logp = ctypes.c_double(0.0)
    nc, ne = ctypes.c_uint64(0), ctypes.c_uint64(0)
    fn = _load().oracle_stochastic_brute if brute else _load().oracle_stochastic_cells
    f64q = ctypes.POINTER(ctypes.c_double)
    _check(fn(p, N, _f(L), _f(b_cand), _f(b_link), _f(alpha), int(seed), int(sample),
              labels.ctypes.data_as(ctypes.POINTER(ctypes.c_int32)), ctypes.byref(logp),
              grad.ctypes.data_as(f64q) if want_grad else None, ctypes.byref(nc), ctypes.byref(ne)))
    return dict(labels=labels[:N], logp=float(logp.value), grad=None if grad is None else grad[:N],
                n_cand=int(nc.value), n_edge=int(ne.value))


def stochastic_edges(pos, L: float, b_cand: float, b_link: float, alpha: float, seed: int, sample: int):
    """Potential edges of one sample (tiny inputs): (ij int32 [P,2], y int32 [P], p float32 [P])."""
    pos, pp = _pos(pos)
    N = pos.shape[0]
    cap = max(1, N * (N - 1) // 2)
    ij = np.empty((cap, 2), np.int32)
    y = np.empty(cap, np.int32)
    pr = np.empty(cap, np.float32)
    i32p = ctypes.POINTER(ctypes.c_int32)
    k = _load().oracle_stochastic_edges(pp, N, _f(L), _f(b_cand), _f(b_link), _f(alpha), int(seed), int(sample), cap,
                                        ij.ctypes.data_as(i32p), y.ctypes.data_as(i32p),
                                        pr.ctypes.data_as(ctypes.POINTER(ctypes.c_float)))
    k = int(_check(k))
    return ij[:k].copy(), y[:k].copy(), pr[:k].copy()


def pref(pos, L: float, b: float) -> int:
    """P_ref: candidate pairs on the tightest grid n_ref = floor(L/b) (metric denominator)."""
    pos, p = _pos(pos)
    P = ctypes.c_uint64(0)
    _check(_load().oracle_pref(p, pos.shape[0], _f(L), _f(b), ctypes.byref(P)))
    return int(P.value)


def linking_length(b_frac: float, L: float, N: int) -> float:
    return float(_load().oracle_linking_length(_f(b_frac), _f(L), int(N)))
