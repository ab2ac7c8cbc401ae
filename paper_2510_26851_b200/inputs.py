"""Seeded synthetic particle sets (the input recipes of DESIGN.md §4).

This module serves BOTH the CPU oracle's tests and the CUDA path's tests/bench, so it
holds none of the method's arithmetic: no linking, no binning, no union-find, no group
reductions.  It only draws random positions with numpy (and, for the Zel'dovich recipe,
one FFT through torch) and casts them to float32.

The recipes stand in for the paper's fastPM 64^3..512^3 snapshots (§2), which
are not available; shapes follow BASELINE.json `configs`, readings #19-#22 of SURVEY.md §8c.
"""
from __future__ import annotations

import math
from dataclasses import dataclass

import numpy as np

SEED_BASE = 268510  # seed = SEED_BASE + config index


@dataclass(frozen=True)
class Workload:
    """One BASELINE.json config made concrete."""

    name: str
    n_side: int          # N = n_side**3
    L: float             # box side
    b_frac: float        # linking length in units of the mean spacing
    N_min: int
    recipe: str          # "clumps" | "nfw" | "zeldovich"
    halos: int = 0
    rms: float = 0.0     # Zel'dovich 3-D rms displacement in units of the spacing
    seed: int = SEED_BASE

    @property
    def N(self) -> int:
        return self.n_side ** 3

    @property
    def spacing(self) -> float:
        return self.L / self.n_side

    @property
    def b(self) -> float:
        """Physical linking length, Eq. 1 evaluated in double, rounded once."""
        return float(np.float32(self.b_frac * self.L / round(self.N ** (1.0 / 3.0))))


# BASELINE.json configs[0..4]; config 4 is a sweep over b_frac on one particle set.
CONFIGS = {
    "cfg0": Workload("cfg0", 32, 1.0, 0.2, 20, "clumps", halos=40, seed=SEED_BASE + 0),
    "cfg1": Workload("cfg1", 128, 1000.0, 0.2, 20, "nfw", halos=20000, seed=SEED_BASE + 1),
    "cfg2": Workload("cfg2", 256, 1000.0, 0.2, 20, "nfw", halos=160000, seed=SEED_BASE + 2),
    "cfg3": Workload("cfg3", 512, 2000.0, 0.2, 20, "zeldovich", rms=0.5, seed=SEED_BASE + 3),
    "cfg4_b0.1": Workload("cfg4_b0.1", 256, 2000.0, 0.1, 20, "zeldovich", rms=1.0, seed=SEED_BASE + 4),
    "cfg4_b0.2": Workload("cfg4_b0.2", 256, 2000.0, 0.2, 20, "zeldovich", rms=1.0, seed=SEED_BASE + 4),
    "cfg4_b0.3": Workload("cfg4_b0.3", 256, 2000.0, 0.3, 20, "zeldovich", rms=1.0, seed=SEED_BASE + 4),
    "cfg4_b0.4": Workload("cfg4_b0.4", 256, 2000.0, 0.4, 20, "zeldovich", rms=1.0, seed=SEED_BASE + 4),
    # NOT a BASELINE.json config.  With P(k) ~ k^-2 the displacement variance sits in the box-scale
    # modes, so at rms = 0.5 .. 1.0 spacing (configs 3 and 4 as specified, reading #20) the density
    # contrast stays at ~0.2 .. 0.3: no shell crossing and almost no pair within 0.4 spacings.  These
    # two push the same recipe past shell crossing (rms 4 spacings) so that the dense-cell and
    # giant-component paths are exercised at full size too.
    "stress_b0.2": Workload("stress_b0.2", 256, 2000.0, 0.2, 20, "zeldovich", rms=4.0, seed=SEED_BASE + 5),
    "stress_b0.4": Workload("stress_b0.4", 256, 2000.0, 0.4, 20, "zeldovich", rms=4.0, seed=SEED_BASE + 5),
}


def scaled(w: Workload, n_side: int, name: str | None = None) -> Workload:
    """Same recipe at another particle count: spacing (and so b) and the halo count per
    particle stay fixed, the box shrinks.  Used for parity cases the oracle finishes fast."""
    f = (n_side / w.n_side)
    return Workload(name or f"{w.name}@{n_side}", n_side, w.L * f, w.b_frac, w.N_min, w.recipe,
                    halos=max(1, int(round(w.halos * f ** 3))) if w.halos else 0, rms=w.rms, seed=w.seed)


def _finish(x: np.ndarray, L: float) -> np.ndarray:
    """float64 -> periodic image in [0, L) -> float32, any value that rounds to >= L set to 0."""
    x = np.mod(x, L)
    x32 = x.astype(np.float32)
    x32[x32 >= np.float32(L)] = 0.0
    return np.ascontiguousarray(x32)


def _iso_dirs(rng: np.random.Generator, m: int) -> np.ndarray:
    v = rng.standard_normal((m, 3))
    v /= np.linalg.norm(v, axis=1, keepdims=True)
    return v


def clump_sizes_pareto(rng: np.random.Generator, halos: int, total: int, floor: int = 20) -> np.ndarray:
    """Reading #22: `halos` Pareto(alpha=1.5) weights scaled to sum `total`, each floored at
    `floor`, the remainder (+/-) given to the largest clump."""
    wgt = rng.pareto(1.5, size=halos) + 1.0
    s = np.floor(wgt / wgt.sum() * total).astype(np.int64)
    s = np.maximum(s, floor)
    s[np.argmax(s)] += total - s.sum()
    assert s.min() >= floor and s.sum() == total
    return s


def make_clumps(w: Workload) -> np.ndarray:
    """G0 (config 0): 70 % uniform + 30 % in isotropic Gaussian clumps, sigma = 0.01 L."""
    rng = np.random.default_rng(w.seed)
    N = w.N
    n_cl = int(round(0.3 * N))
    sizes = clump_sizes_pareto(rng, w.halos, n_cl)
    bg = rng.random((N - n_cl, 3)) * w.L
    centres = rng.random((w.halos, 3)) * w.L
    mem = np.repeat(centres, sizes, axis=0) + rng.standard_normal((n_cl, 3)) * (0.01 * w.L)
    return _finish(np.concatenate([bg, mem], axis=0), w.L)


def _mmax_for_mean(mean: float, lo: float = 20.0, slope: float = 1.9) -> float:
    """Solve the upper cut of dn/dM ~ M^-slope on [lo, M_max] so that E[M] = mean (reading #21)."""
    def mean_of(mx: float) -> float:
        a = 1.0 - slope   # exponent of the integral of the pdf
        c = 2.0 - slope   # exponent of the integral of M * pdf
        return ((mx ** c - lo ** c) / c) / ((mx ** a - lo ** a) / a)
    a_, b_ = lo * 1.0001, lo * 1e4
    for _ in range(200):
        mid = 0.5 * (a_ + b_)
        if mean_of(mid) < mean:
            a_ = mid
        else:
            b_ = mid
    return 0.5 * (a_ + b_)


def halo_member_counts(rng: np.random.Generator, halos: int, target_total: int) -> np.ndarray:
    """Power-law mass function, slope -1.9, min 20, truncated so the mean matches; draws are
    rounded down (the caller fixes the total through the background count)."""
    lo, slope = 20.0, 1.9
    mx = _mmax_for_mean(target_total / halos, lo, slope)
    a = 1.0 - slope
    u = rng.random(halos)
    m = (lo ** a + u * (mx ** a - lo ** a)) ** (1.0 / a)
    return np.floor(m).astype(np.int64)


def make_nfw(w: Workload) -> np.ndarray:
    """G1 (configs 1, 2): 60 % uniform background + 40 % in NFW-like halos.
    radial CDF ~ ln(1+x) - x/(1+x), x = r/r_s <= c;  r_s = b * 10^U(log10 .05, log10 .5);
    c ~ U(5, 15); isotropic directions; centres uniform."""
    rng = np.random.default_rng(w.seed)
    N, H, b = w.N, w.halos, w.b
    counts = halo_member_counts(rng, H, int(round(0.4 * N)))
    n_mem = int(counts.sum())
    bg = rng.random((N - n_mem, 3)) * w.L
    centres = rng.random((H, 3)) * w.L
    r_s = b * 10.0 ** rng.uniform(math.log10(0.05), math.log10(0.5), size=H)
    conc = rng.uniform(5.0, 15.0, size=H)
    xt = np.linspace(0.0, 15.0, 30001)
    mt = np.log1p(xt) - xt / (1.0 + xt)
    m_c = np.log1p(conc) - conc / (1.0 + conc)
    u = rng.random(n_mem) * np.repeat(m_c, counts)
    x = np.interp(u, mt, xt)
    r = x * np.repeat(r_s, counts)
    mem = np.repeat(centres, counts, axis=0) + _iso_dirs(rng, n_mem) * r[:, None]
    return _finish(np.concatenate([bg, mem], axis=0), w.L)


def make_zeldovich(w: Workload, device: str = "cpu") -> np.ndarray:
    """G3 (configs 3, 4): lattice q displaced by psi = grad^-1 of a Gaussian field with
    P(k) ~ k^-2:  psi_k = i k delta_k / k^2, scaled so sqrt(mean(psi.psi)) = rms * spacing.
    White noise comes from numpy (seeded); the FFTs run through torch on `device`."""
    import torch

    n, L = w.n_side, w.L
    rng = np.random.default_rng(w.seed)
    real = torch.float32 if n >= 512 else torch.float64
    white = torch.from_numpy(rng.standard_normal((n, n, n), dtype=np.float32 if n >= 512 else np.float64)).to(device)
    dk = torch.fft.rfftn(white)
    del white
    kf = torch.fft.fftfreq(n, d=1.0 / n, device=device, dtype=real)
    kr = torch.fft.rfftfreq(n, d=1.0 / n, device=device, dtype=real)
    k2 = kf[:, None, None] ** 2 + kf[None, :, None] ** 2 + kr[None, None, :] ** 2
    k2[0, 0, 0] = 1.0
    # delta_k = white_k * sqrt(P) = white_k / k ;  psi_k = i k_vec delta_k / k^2
    base = dk * k2.pow(-1.5)
    base[0, 0, 0] = 0.0
    del dk, k2
    comps = []
    for ax, kv in enumerate((kf[:, None, None], kf[None, :, None], kr[None, None, :])):
        psi = torch.fft.irfftn(1j * kv * base, s=(n, n, n))
        comps.append(psi)
    del base
    ms = sum(float((c.double() ** 2).mean()) for c in comps)
    scale = w.rms * w.spacing / math.sqrt(ms)
    q = (torch.arange(n, device=device, dtype=torch.float64) + 0.5) * w.spacing
    out = np.empty((n ** 3, 3), dtype=np.float32)
    grids = (q[:, None, None], q[None, :, None], q[None, None, :])
    for ax in range(3):
        x = (grids[ax] + comps[ax].double() * scale).expand(n, n, n).reshape(-1)
        x = torch.remainder(x, L).float()
        x[x >= L] = 0.0
        out[:, ax] = x.cpu().numpy()
        comps[ax] = None
    return out


def make_positions(w: Workload, device: str = "cpu") -> np.ndarray:
    """[N, 3] float32 positions in [0, L) for a workload."""
    if w.recipe == "clumps":
        return make_clumps(w)
    if w.recipe == "nfw":
        return make_nfw(w)
    if w.recipe == "zeldovich":
        return make_zeldovich(w, device)
    raise ValueError(w.recipe)


def make_masses(w: Workload) -> np.ndarray:
    """uniform(0.5, 1.5) float32 masses (the second run per config that exercises H8)."""
    rng = np.random.default_rng(w.seed + 7919)
    return rng.uniform(0.5, 1.5, size=w.N).astype(np.float32)


# ----------------------------------------------------------------------------------------------
# small constructed inputs used by the closed-form pins (SURVEY.md §8c "Closed forms")
# ----------------------------------------------------------------------------------------------

def lattice(n: int, L: float) -> np.ndarray:
    """n^3 points at (i + 0) * L/n  — dyadic when L and n are powers of two."""
    g = (np.arange(n, dtype=np.float64)) * (L / n)
    x, y, z = np.meshgrid(g, g, g, indexing="ij")
    return np.ascontiguousarray(np.stack([x.ravel(), y.ravel(), z.ravel()], axis=1).astype(np.float32))


def planted_cliques(seed: int, sizes, L: float, b: float, grid_side: int | None = None):
    """Clumps whose members all lie within 0.45 b of a centre; centres sit on distinct nodes of a
    coarse lattice with pitch >= 4 b (so min-image centre distance > 3 b).  Members are shuffled.
    Returns (pos float32 [N,3], clump id per particle)."""
    rng = np.random.default_rng(seed)
    sizes = np.asarray(sizes, dtype=np.int64)
    K = len(sizes)
    g = grid_side or int(math.floor(L / (4.0 * b)))
    assert g ** 3 >= K, "box too small for that many separated clumps"
    nodes = rng.choice(g ** 3, size=K, replace=False)
    pitch = L / g
    centres = np.stack([nodes % g, (nodes // g) % g, nodes // (g * g)], axis=1) * pitch + 0.5 * pitch
    n = int(sizes.sum())
    rad = 0.45 * b * rng.random(n) ** (1.0 / 3.0)
    pts = np.repeat(centres, sizes, axis=0) + _iso_dirs(rng, n) * rad[:, None]
    ids = np.repeat(np.arange(K), sizes)
    perm = rng.permutation(n)
    return _finish(pts[perm], L), ids[perm]


def chain(n: int, L: float) -> np.ndarray:
    """n points equally spaced along x through the whole periodic box (y = z = L/4)."""
    x = np.arange(n, dtype=np.float64) * (L / n)
    return _finish(np.stack([x, np.full(n, L / 4), np.full(n, L / 4)], axis=1), L)
