"""Thin Python binding over the C ABI of include/fof.h: argument marshalling only.

Every step of the path runs inside libfof_b200.so; PyTorch is used for device memory, pinned
host memory and streams.  The module-level functions carry the C names (fof_create, fof_link,
fof_groups, ...); `FoF` is a small convenience object that owns the handle and the workspace.
"""
from __future__ import annotations

import ctypes
import os

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libfof_b200.so")

FOF_OK = 0
FOF_ERR_INVALID_ARG = -1
FOF_ERR_UNSUPPORTED = -2
FOF_ERR_CUDA = -3
FOF_ERR_NONFINITE = -4
FOF_ERR_CAPACITY = -5
FOF_ERR_STATE = -6

_lib = None


class FofError(RuntimeError):
    def __init__(self, code: int, msg: str):
        super().__init__(f"fof error {code}: {msg}")
        self.code = code


def lib():
    """Load libfof_b200.so (built by `python -m paper_2510_26851_b200.build`); fail loudly if absent."""
    global _lib
    if _lib is None:
        if not os.path.exists(LIB_PATH):
            raise ImportError(
                f"{LIB_PATH} is missing: build it with `python -m paper_2510_26851_b200.build` "
                "(nvcc, sm_100a). There is no CPU fallback.")
        L = ctypes.CDLL(LIB_PATH)
        vp, i64, i32, f32 = ctypes.c_void_p, ctypes.c_int64, ctypes.c_int32, ctypes.c_float
        L.fof_linking_length.restype = f32
        L.fof_linking_length.argtypes = [f32, f32, i64]
        L.fof_create.restype = ctypes.c_int
        L.fof_create.argtypes = [i64, f32, f32, i32, ctypes.POINTER(vp)]
        L.fof_destroy.restype = None
        L.fof_destroy.argtypes = [vp]
        L.fof_set_grid.restype = ctypes.c_int
        L.fof_set_grid.argtypes = [vp, i32]
        L.fof_get_grid.restype = ctypes.c_int
        L.fof_get_grid.argtypes = [vp, ctypes.POINTER(i32), ctypes.POINTER(i64), ctypes.POINTER(i32)]
        L.fof_set_path.restype = ctypes.c_int
        L.fof_set_path.argtypes = [vp, i32]
        L.fof_link_path.restype = ctypes.c_int
        L.fof_link_path.argtypes = [vp, vp, vp, ctypes.POINTER(i32), ctypes.POINTER(i32), ctypes.POINTER(i32)]
        L.fof_workspace_bytes.restype = ctypes.c_size_t
        L.fof_workspace_bytes.argtypes = [vp]
        L.fof_link.restype = ctypes.c_int
        L.fof_link.argtypes = [vp, vp, vp, vp, vp]
        L.fof_link_stats.restype = ctypes.c_int
        L.fof_link_stats.argtypes = [vp, vp, vp, ctypes.POINTER(ctypes.c_uint64), ctypes.POINTER(ctypes.c_uint64),
                                     ctypes.POINTER(ctypes.c_uint64)]
        L.fof_groups.restype = ctypes.c_int
        L.fof_groups.argtypes = [vp, vp, vp, vp, vp, vp, vp, vp, vp, vp, i64, ctypes.POINTER(i64), vp]
        L.fof_link_stochastic.restype = ctypes.c_int
        L.fof_link_stochastic.argtypes = [vp, f32, f32, ctypes.c_uint64, ctypes.c_uint32, vp, vp, vp, vp, vp]
        L.fof_stochastic_scratch_bytes.restype = ctypes.c_size_t
        L.fof_stochastic_scratch_bytes.argtypes = [vp, ctypes.c_int32]
        L.fof_link_stochastic_batch.restype = ctypes.c_int
        L.fof_link_stochastic_batch.argtypes = [vp, f32, f32, ctypes.c_uint64, ctypes.c_uint32, ctypes.c_int32, vp, vp, vp,
                                                vp, vp, vp]
        L.fof_stochastic_list_bytes.restype = ctypes.c_size_t
        L.fof_stochastic_list_bytes.argtypes = [vp, ctypes.c_uint64]
        L.fof_stochastic_list_build.restype = ctypes.c_int
        L.fof_stochastic_list_build.argtypes = [vp, f32, f32, vp, ctypes.c_size_t, ctypes.POINTER(ctypes.c_uint64), vp, vp]
        L.fof_link_stochastic_list.restype = ctypes.c_int
        L.fof_link_stochastic_list.argtypes = [vp, vp, ctypes.c_uint64, ctypes.c_uint32, ctypes.c_int32, vp, vp, vp, vp,
                                               vp, vp]
        L.fof_subgroups.restype = ctypes.c_int
        L.fof_subgroups.argtypes = [vp, vp, vp, vp, vp, i64, f32, f32, f32, vp, vp, vp]
        L.fof_layer_select.restype = ctypes.c_int
        L.fof_layer_select.argtypes = [vp, i64, f32, i32, f32, f32, vp, vp, vp]
        L.fof_component_min.restype = ctypes.c_int
        L.fof_component_min.argtypes = [vp, vp, i64, vp, vp, vp]
        L.fof_merge_labels.restype = ctypes.c_int
        L.fof_merge_labels.argtypes = [vp, i64, vp, i64, vp, i64, vp]
        L.fof_merge_labels_sparse.restype = ctypes.c_int
        L.fof_merge_labels_sparse.argtypes = [vp, i64, vp, i64, vp, vp, i64, vp]
        L.fof_combine_groups.restype = ctypes.c_int
        L.fof_combine_groups.argtypes = [vp, i64, vp, f32, vp, i64, vp, vp, vp, vp, vp, vp, vp]
        L.fof_group_sigma.restype = ctypes.c_int
        L.fof_group_sigma.argtypes = [vp, vp, vp, vp, vp, vp, i64, vp, vp, vp]
        L.fof_group_sigma_static.restype = ctypes.c_int
        L.fof_group_sigma_static.argtypes = [vp, vp, vp, vp, vp, vp, i64, vp, vp]
        L.fof_groups_backward.restype = ctypes.c_int
        L.fof_groups_backward.argtypes = [vp, vp, vp, vp, vp, vp, vp, vp, vp, i64, vp, vp]
        L.fof_host_device_bytes.restype = ctypes.c_size_t
        L.fof_host_device_bytes.argtypes = [vp, i64]
        L.fof_host_submit.restype = ctypes.c_int
        L.fof_host_submit.argtypes = [vp, ctypes.c_int32, vp, vp, vp, vp, vp, vp, vp, vp, i64, vp]
        L.fof_host_wait.restype = ctypes.c_int
        L.fof_host_wait.argtypes = [vp, ctypes.c_int32, ctypes.POINTER(i64)]
        L.fof_run_host.restype = ctypes.c_int
        L.fof_run_host.argtypes = [vp, vp, vp, vp, vp, vp, vp, vp, vp, i64, ctypes.POINTER(i64), vp, vp]
        L.fof_status.restype = ctypes.c_int
        L.fof_status.argtypes = [vp, vp, vp]
        L.fof_profile_enable.restype = ctypes.c_int
        L.fof_profile_enable.argtypes = [vp, ctypes.c_int]
        L.fof_profile_only.restype = ctypes.c_int
        L.fof_profile_only.argtypes = [vp, ctypes.c_int]
        L.fof_profile_count.restype = ctypes.c_int
        L.fof_profile_count.argtypes = [vp]
        L.fof_profile_name.restype = ctypes.c_char_p
        L.fof_profile_name.argtypes = [vp, ctypes.c_int]
        L.fof_profile_read.restype = ctypes.c_int
        L.fof_profile_read.argtypes = [vp, ctypes.POINTER(ctypes.c_float), ctypes.c_int]
        L.fof_launch_count.restype = ctypes.c_uint64
        L.fof_launch_count.argtypes = [vp]
        L.fof_measure_fp32_issue.restype = ctypes.c_int
        L.fof_measure_fp32_issue.argtypes = [ctypes.POINTER(ctypes.c_double), vp]
        L.fof_measure_scatter.restype = ctypes.c_int
        L.fof_measure_scatter.argtypes = [vp, vp, i64, i32, i32, ctypes.POINTER(ctypes.c_double), vp]
        L.fof_error_string.restype = ctypes.c_char_p
        L.fof_error_string.argtypes = [ctypes.c_int]
        L.fof_last_cuda_error.restype = ctypes.c_char_p
        L.fof_last_cuda_error.argtypes = [vp]
        _lib = L
    return _lib


def _f(x) -> float:
    return float(np.float32(x))


def _check(rc: int, handle=None):
    if rc != FOF_OK:
        msg = lib().fof_error_string(rc).decode()
        if rc == FOF_ERR_CUDA and handle is not None:
            msg += " (" + lib().fof_last_cuda_error(handle).decode() + ")"
        raise FofError(rc, msg)


def _ptr(t):
    return None if t is None else ctypes.c_void_p(t.data_ptr())


def _stream_ptr(stream):
    import torch

    s = stream if stream is not None else torch.cuda.current_stream()
    return ctypes.c_void_p(s.cuda_stream)


# ---------------------------------------------------------------- C-named functions
def fof_linking_length(b_frac: float, L: float, N: int) -> float:
    return float(lib().fof_linking_length(_f(b_frac), _f(L), int(N)))


def fof_create(N: int, L: float, b: float, N_min: int):
    h = ctypes.c_void_p()
    _check(lib().fof_create(int(N), _f(L), _f(b), int(N_min), ctypes.byref(h)))
    return h


def fof_destroy(h):
    lib().fof_destroy(h)


def fof_set_grid(h, n: int):
    _check(lib().fof_set_grid(h, int(n)))


def fof_get_grid(h):
    n, c, m = ctypes.c_int32(), ctypes.c_int64(), ctypes.c_int32()
    _check(lib().fof_get_grid(h, ctypes.byref(n), ctypes.byref(c), ctypes.byref(m)))
    return n.value, c.value, m.value


FOF_PATH_AUTO, FOF_PATH_CELLS, FOF_PATH_BLOCKS = 0, 1, 2
_PATHS = {"auto": FOF_PATH_AUTO, "cells": FOF_PATH_CELLS, "blocks": FOF_PATH_BLOCKS}


def fof_set_path(h, path):
    """path: "auto", "cells" (always the cell path) or "blocks" (block path where the plan admits it)."""
    _check(lib().fof_set_path(h, _PATHS[path] if isinstance(path, str) else int(path)))


def fof_link_path(h, ws, stream=None):
    """("blocks" | "cells" = what the last fof_link ran, blocks of the plan, records of the fullest block)"""
    p, nb, mb = ctypes.c_int32(), ctypes.c_int32(), ctypes.c_int32()
    _check(lib().fof_link_path(h, _ptr(ws), _stream_ptr(stream), ctypes.byref(p), ctypes.byref(nb), ctypes.byref(mb)), h)
    return ("blocks" if p.value == FOF_PATH_BLOCKS else "cells"), int(nb.value), int(mb.value)


def fof_workspace_bytes(h) -> int:
    return int(lib().fof_workspace_bytes(h))


def fof_link(h, pos, labels, ws, stream=None):
    """pos: cuda float32 [N,3] contiguous; labels: cuda int32 [N]; ws: cuda uint8 workspace."""
    _check(lib().fof_link(h, _ptr(pos), _ptr(labels), _ptr(ws), _stream_ptr(stream)), h)


def fof_link_stats(h, ws, stream=None):
    """(true edges E, distance tests executed, candidate pairs of the unfiltered stencil on this grid)"""
    e, t, gp = ctypes.c_uint64(), ctypes.c_uint64(), ctypes.c_uint64()
    _check(lib().fof_link_stats(h, _ptr(ws), _stream_ptr(stream), ctypes.byref(e), ctypes.byref(t),
                                ctypes.byref(gp)), h)
    return int(e.value), int(t.value), int(gp.value)


def fof_groups(h, pos, mass, labels, ws, group_label, group_size, group_mass, group_com, particle_group, cap,
               stream=None) -> int:
    K = ctypes.c_int64()
    _check(lib().fof_groups(h, _ptr(pos), _ptr(mass), _ptr(labels), _ptr(ws), _ptr(group_label), _ptr(group_size),
                            _ptr(group_mass), _ptr(group_com), _ptr(particle_group), int(cap), ctypes.byref(K),
                            _stream_ptr(stream)), h)
    return int(K.value)


def fof_link_stochastic(h, b_link, alpha, seed, sample, labels, logp, grad_pos, ws, stream=None):
    """labels: cuda int32 [N]; logp: cuda float64 [1]; grad_pos: cuda float32 [N,3] or None."""
    _check(lib().fof_link_stochastic(h, _f(b_link), _f(alpha), int(seed), int(sample), _ptr(labels), _ptr(logp),
                                     _ptr(grad_pos), _ptr(ws), _stream_ptr(stream)), h)


def fof_stochastic_scratch_bytes(h, S):
    return int(lib().fof_stochastic_scratch_bytes(h, int(S)))


def fof_link_stochastic_batch(h, b_link, alpha, seed, sample, S, labels, logp, grad_pos, scratch, ws, stream=None):
    """labels: cuda int32 [S,N]; logp: cuda float64 [S]; grad_pos: cuda float32 [S,N,3] or None; scratch: cuda bytes."""
    _check(lib().fof_link_stochastic_batch(h, _f(b_link), _f(alpha), int(seed), int(sample), int(S), _ptr(labels),
                                           _ptr(logp), _ptr(grad_pos), _ptr(scratch), _ptr(ws), _stream_ptr(stream)), h)


def fof_stochastic_list_bytes(h, records: int) -> int:
    return int(lib().fof_stochastic_list_bytes(h, int(records)))


def fof_stochastic_list_build(h, b_link, alpha, list_buf, ws, stream=None):
    """list_buf: cuda uint8 tensor.  Returns (records, filled): filled is False if list_buf was too small for them."""
    R = ctypes.c_uint64()
    rc = lib().fof_stochastic_list_build(h, _f(b_link), _f(alpha), _ptr(list_buf), int(list_buf.numel()),
                                         ctypes.byref(R), _ptr(ws), _stream_ptr(stream))
    if rc == FOF_ERR_CAPACITY and R.value <= 0xFFFFFFFF:
        return int(R.value), False
    _check(rc, h)
    return int(R.value), True


def fof_link_stochastic_list(h, list_buf, seed, sample, S, labels, logp, grad_pos, scratch, ws, stream=None):
    """labels: cuda int32 [S,N]; logp: cuda float64 [S]; grad_pos: cuda float32 [S,N,3] or None; scratch: cuda bytes."""
    _check(lib().fof_link_stochastic_list(h, _ptr(list_buf), int(seed), int(sample), int(S), _ptr(labels), _ptr(logp),
                                          _ptr(grad_pos), _ptr(scratch), _ptr(ws), _stream_ptr(stream)), h)


def fof_subgroups(h, pos, vel, particle_group, group_size, K, sigma_x, sigma_v, ell, sub_labels, ws, stream=None):
    _check(lib().fof_subgroups(h, _ptr(pos), _ptr(vel), _ptr(particle_group), _ptr(group_size), int(K), _f(sigma_x),
                               _f(sigma_v), _f(ell), _ptr(sub_labels), _ptr(ws), _stream_ptr(stream)), h)


def fof_layer_select(pos, L, axis, lo, width, out_idx, count, stream=None):
    _check(lib().fof_layer_select(_ptr(pos), int(pos.shape[0]), _f(L), int(axis), _f(lo), _f(width), _ptr(out_idx),
                                  _ptr(count), _stream_ptr(stream)))


def fof_component_min(labels, ids, tmp, out, stream=None):
    _check(lib().fof_component_min(_ptr(labels), _ptr(ids), int(labels.shape[0]), _ptr(tmp), _ptr(out),
                                   _stream_ptr(stream)))


def fof_merge_labels(pairs, parent, labels, stream=None):
    _check(lib().fof_merge_labels(_ptr(pairs), int(pairs.shape[0]), _ptr(parent), int(parent.shape[0]), _ptr(labels),
                                  int(labels.shape[0]), _stream_ptr(stream)))


def fof_merge_labels_sparse(pairs, uniq, parent, labels, stream=None):
    """pairs: cuda int32 [P,2]; uniq: cuda int32 [U] ascending distinct labels of the pairs; parent: scratch [U]."""
    _check(lib().fof_merge_labels_sparse(_ptr(pairs), int(pairs.shape[0]), _ptr(uniq), int(uniq.shape[0]), _ptr(parent),
                                         _ptr(labels), int(labels.shape[0]), _stream_ptr(stream)))


def fof_combine_groups(want, ref, L, part_label, part_size, part_mass, part_com, out_size, out_mass, out_com, stream=None):
    _check(lib().fof_combine_groups(_ptr(want), int(want.shape[0]), _ptr(ref), _f(L), _ptr(part_label),
                                    int(part_label.shape[0]), _ptr(part_size), _ptr(part_mass), _ptr(part_com),
                                    _ptr(out_size), _ptr(out_mass), _ptr(out_com), _stream_ptr(stream)))


def fof_group_sigma(h, pos, mass, particle_group, group_mass, group_com, K, ws, group_sigma, stream=None):
    _check(lib().fof_group_sigma(h, _ptr(pos), _ptr(mass), _ptr(particle_group), _ptr(group_mass), _ptr(group_com),
                                 int(K), _ptr(ws), _ptr(group_sigma), _stream_ptr(stream)), h)


FOF_SIGMA_STATIC_MAX_GROUPS = 262144


def fof_group_sigma_static(h, pos, mass, particle_group, group_mass, group_com, K, group_sigma, stream=None):
    """fof_group_sigma with the library's static scratch instead of a workspace (K <= FOF_SIGMA_STATIC_MAX_GROUPS)."""
    _check(lib().fof_group_sigma_static(h, _ptr(pos), _ptr(mass), _ptr(particle_group), _ptr(group_mass),
                                        _ptr(group_com), int(K), _ptr(group_sigma), _stream_ptr(stream)), h)


def fof_groups_backward(h, pos, mass, particle_group, group_mass, group_com, group_sigma, grad_com, grad_sigma, K,
                        grad_pos, stream=None):
    _check(lib().fof_groups_backward(h, _ptr(pos), _ptr(mass), _ptr(particle_group), _ptr(group_mass),
                                     _ptr(group_com), _ptr(group_sigma), _ptr(grad_com), _ptr(grad_sigma), int(K),
                                     _ptr(grad_pos), _stream_ptr(stream)), h)


def fof_host_device_bytes(h, cap: int) -> int:
    return int(lib().fof_host_device_bytes(h, int(cap)))


def fof_run_host(h, pos_host, mass_host, labels_host, group_label_host, group_size_host, group_mass_host,
                 group_com_host, particle_group_host, cap, dev_buf, stream=None) -> int:
    """All *_host are CPU tensors (pinned for speed); dev_buf is a cuda uint8 tensor."""
    K = ctypes.c_int64()
    _check(lib().fof_run_host(h, _ptr(pos_host), _ptr(mass_host), _ptr(labels_host), _ptr(group_label_host),
                              _ptr(group_size_host), _ptr(group_mass_host), _ptr(group_com_host),
                              _ptr(particle_group_host), int(cap), ctypes.byref(K), _ptr(dev_buf),
                              _stream_ptr(stream)), h)
    return int(K.value)


def fof_host_submit(h, slot, pos_host, mass_host, labels_host, group_label_host, group_size_host, group_mass_host,
                    group_com_host, particle_group_host, cap, dev_buf):
    """Enqueue half of fof_run_host (slot 0 or 1, each with its own dev_buf); pinned host tensors."""
    _check(lib().fof_host_submit(h, int(slot), _ptr(pos_host), _ptr(mass_host), _ptr(labels_host),
                                 _ptr(group_label_host), _ptr(group_size_host), _ptr(group_mass_host),
                                 _ptr(group_com_host), _ptr(particle_group_host), int(cap), _ptr(dev_buf)), h)


def fof_host_wait(h, slot) -> int:
    """Completion half: blocks until the slot's results are in the host buffers; returns K."""
    K = ctypes.c_int64()
    _check(lib().fof_host_wait(h, int(slot), ctypes.byref(K)), h)
    return int(K.value)


def fof_status(h, ws, stream=None) -> int:
    return int(lib().fof_status(h, _ptr(ws), _stream_ptr(stream)))


def fof_profile_enable(h, slots: int):
    _check(lib().fof_profile_enable(h, int(slots)), h)


def fof_profile_only(h, stage_name=None):
    """Record events for one stage only (by name), or for every stage (None)."""
    k = -1 if stage_name is None else fof_profile_names(h).index(stage_name)
    _check(lib().fof_profile_only(h, k), h)


def fof_profile_names(h):
    n = lib().fof_profile_count(h)
    return [lib().fof_profile_name(h, k).decode() for k in range(n)]


def fof_profile_read(h):
    """{stage name: mean device milliseconds} over the steps recorded since the last read."""
    n = lib().fof_profile_count(h)
    buf = (ctypes.c_float * n)()
    _check(lib().fof_profile_read(h, buf, n), h)
    return {lib().fof_profile_name(h, k).decode(): float(buf[k]) for k in range(n)}


def fof_measure_fp32_issue(stream=None) -> float:
    """FP32 lane-operations per second on a non-FMA FADD + FMUL stream (measured ceiling of the link predicate)."""
    v = ctypes.c_double()
    _check(lib().fof_measure_fp32_issue(ctypes.byref(v), _stream_ptr(stream)))
    return float(v.value)


def fof_measure_scatter(src, dst, log2_window: int, scatter_stores: bool, stream=None) -> float:
    """records/s of a copy of 16-byte records whose stores (or loads) are scattered inside 2^k-record windows."""
    v = ctypes.c_double()
    n = src.numel() * src.element_size() // 16
    _check(lib().fof_measure_scatter(_ptr(src), _ptr(dst), int(n), int(log2_window), int(bool(scatter_stores)),
                                     ctypes.byref(v), _stream_ptr(stream)))
    return float(v.value)


def fof_launch_count(h) -> int:
    return int(lib().fof_launch_count(h))


# ---------------------------------------------------------------- convenience object
class FoF:
    """Owns a plan handle and its device workspace (torch uint8 tensor)."""

    def __init__(self, N: int, L: float, b: float, N_min: int = 20, device="cuda:0", grid: int | None = None,
                 path: str = "auto"):
        import torch

        if not torch.cuda.is_available():
            raise RuntimeError("paper_2510_26851_b200 needs a CUDA device: there is no CPU fallback")
        self.N, self.L, self.b, self.N_min = int(N), _f(L), _f(b), int(N_min)
        self.device = torch.device(device)
        self.h = fof_create(N, L, b, N_min)
        if grid is not None:
            fof_set_grid(self.h, grid)
        if path != "auto":
            fof_set_path(self.h, path)
        self.cap = max(1, self.N // self.N_min)
        with torch.cuda.device(self.device):
            self.ws = torch.empty(fof_workspace_bytes(self.h) + 256, dtype=torch.uint8, device=self.device)
        assert self.ws.data_ptr() % 256 == 0

    @property
    def grid(self):
        return fof_get_grid(self.h)

    def close(self):
        if getattr(self, "h", None) is not None:
            fof_destroy(self.h)
            self.h = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def link(self, pos, labels=None, stream=None):
        import torch

        assert pos.is_cuda and pos.dtype == torch.float32 and pos.is_contiguous() and pos.shape == (self.N, 3)
        if labels is None:
            labels = torch.empty(self.N, dtype=torch.int32, device=pos.device)
        with torch.cuda.device(self.device):
            fof_link(self.h, pos, labels, self.ws, stream)
        return labels

    def link_stats(self, stream=None):
        with __import__("torch").cuda.device(self.device):
            return fof_link_stats(self.h, self.ws, stream)

    def link_path(self, stream=None):
        with __import__("torch").cuda.device(self.device):
            return fof_link_path(self.h, self.ws, stream)

    def status(self, stream=None) -> int:
        with __import__("torch").cuda.device(self.device):
            return fof_status(self.h, self.ws, stream)

    def alloc_groups(self, cap=None, particle_group=False):
        import torch

        cap = self.cap if cap is None else int(cap)
        d = self.device
        out = dict(cap=cap,
                   group_label=torch.empty(cap, dtype=torch.int32, device=d),
                   group_size=torch.empty(cap, dtype=torch.int32, device=d),
                   group_mass=torch.empty(cap, dtype=torch.float32, device=d),
                   group_com=torch.empty((cap, 3), dtype=torch.float32, device=d),
                   particle_group=torch.empty(self.N, dtype=torch.int32, device=d) if particle_group else None)
        return out

    def link_stochastic(self, b_link, alpha, seed, sample, want_grad=True, stream=None):
        """One stochastic-edge sample on the binning of the last link(): (labels, logp tensor, grad or None)."""
        import torch

        d = self.device
        labels = torch.empty(self.N, dtype=torch.int32, device=d)
        logp = torch.zeros(1, dtype=torch.float64, device=d)
        grad = torch.empty((self.N, 3), dtype=torch.float32, device=d) if want_grad else None
        with torch.cuda.device(d):
            fof_link_stochastic(self.h, b_link, alpha, seed, sample, labels, logp, grad, self.ws, stream)
        return labels, logp, grad

    def link_stochastic_batch(self, b_link, alpha, seed, sample, S, want_grad=True, stream=None):
        """S samples sample .. sample + S - 1 in one call: (labels [S,N], logp [S], grad [S,N,3] or None)."""
        import torch

        d = self.device
        labels = torch.empty((S, self.N), dtype=torch.int32, device=d)
        logp = torch.zeros(S, dtype=torch.float64, device=d)
        grad = torch.empty((S, self.N, 3), dtype=torch.float32, device=d) if want_grad else None
        scratch = torch.empty(max(fof_stochastic_scratch_bytes(self.h, S), 4), dtype=torch.uint8, device=d)
        with torch.cuda.device(d):
            fof_link_stochastic_batch(self.h, b_link, alpha, seed, sample, S, labels, logp, grad, scratch, self.ws, stream)
        return labels, logp, grad

    def stochastic_list(self, b_link, alpha, stream=None):
        """The potential-edge list of the last link() (a cuda byte tensor to pass to link_stochastic_list) and its
        number of records; two calls of the build: the first one sizes the buffer."""
        import torch

        d = self.device
        with torch.cuda.device(d):
            buf = torch.empty(fof_stochastic_list_bytes(self.h, 0), dtype=torch.uint8, device=d)
            records, filled = fof_stochastic_list_build(self.h, b_link, alpha, buf, self.ws, stream)
            if not filled:
                del buf
                buf = torch.empty(fof_stochastic_list_bytes(self.h, records), dtype=torch.uint8, device=d)
                records, filled = fof_stochastic_list_build(self.h, b_link, alpha, buf, self.ws, stream)
                assert filled
        assert buf.data_ptr() % 256 == 0
        return buf, records

    def link_stochastic_list(self, slist, seed, sample, S, want_grad=True, stream=None):
        """S samples over the list of stochastic_list(): (labels [S,N], logp [S], grad [S,N,3] or None)."""
        import torch

        d = self.device
        labels = torch.empty((S, self.N), dtype=torch.int32, device=d)
        logp = torch.zeros(S, dtype=torch.float64, device=d)
        grad = torch.empty((S, self.N, 3), dtype=torch.float32, device=d) if want_grad else None
        scratch = torch.empty(max(fof_stochastic_scratch_bytes(self.h, S), 4), dtype=torch.uint8, device=d)
        with torch.cuda.device(d):
            fof_link_stochastic_list(self.h, slist, seed, sample, S, labels, logp, grad, scratch, self.ws, stream)
        return labels, logp, grad

    def subgroups(self, pos, vel, g, sigma_x, sigma_v, ell, stream=None):
        """6-D sub-halo labels [N] inside the groups `g` returned by groups(..., particle_group=True)."""
        import torch

        sub = torch.empty(self.N, dtype=torch.int32, device=pos.device)
        with torch.cuda.device(self.device):
            fof_subgroups(self.h, pos, vel, g["particle_group"], g["group_size"], g["K"], sigma_x, sigma_v, ell, sub,
                          self.ws, stream)
        return sub

    def group_sigma(self, pos, g, mass=None, stream=None):
        """Halo decoration sigma [K] of the groups `g` returned by groups(..., particle_group=True)."""
        import torch

        K = g["K"]
        sig = torch.empty(K, dtype=torch.float32, device=pos.device)
        with torch.cuda.device(self.device):
            fof_group_sigma(self.h, pos, mass, g["particle_group"], g["group_mass"], g["group_com"], K, self.ws, sig,
                            stream)
        return sig

    def groups_backward(self, pos, g, grad_com=None, group_sigma=None, grad_sigma=None, mass=None, stream=None):
        """Frozen-assignment backward: grad_pos [N,3] from dL/dX [K,3] (and dL/dsigma [K])."""
        import torch

        out = torch.empty((self.N, 3), dtype=torch.float32, device=pos.device)
        with torch.cuda.device(self.device):
            fof_groups_backward(self.h, pos, mass, g["particle_group"], g["group_mass"], g["group_com"], group_sigma,
                                grad_com, grad_sigma, g["K"], out, stream)
        return out

    def groups(self, pos, labels, mass=None, out=None, particle_group=False, stream=None):
        """Returns dict(K, group_label[:K], group_size[:K], group_mass[:K], group_com[:K], particle_group)."""
        import torch

        if out is None:
            out = self.alloc_groups(particle_group=particle_group)
        with torch.cuda.device(self.device):
            K = fof_groups(self.h, pos, mass, labels, self.ws, out["group_label"], out["group_size"],
                           out["group_mass"], out["group_com"], out["particle_group"], out["cap"], stream)
        return dict(K=K, group_label=out["group_label"][:K], group_size=out["group_size"][:K],
                    group_mass=out["group_mass"][:K], group_com=out["group_com"][:K],
                    particle_group=out["particle_group"])
