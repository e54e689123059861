"""The five synthetic workloads of BASELINE.json / SURVEY.md §8(d).

They take the shapes, sizes and value structure of the paper's problems
(PAPER.md:128-136 PWR assembly; PAPER.md:164-166 criticality accident) and stand
in for them: the paper's MCATK models and ACE cross-section libraries are not
available, and nothing of them is reproduced here.

Rules:
  * one PCG64 stream per (config, stream, batch): SeedSequence([1706074760,
    config, stream, batch]); stream 0 = mesh/materials, 1..M = tables, 9 = rays;
    uniforms are numpy's (bits >> 11) * 2**-53.
  * every array the mixed-precision library stores in fp32 (energy grids, sigma
    tables, ray fields, densities, fractions) is rounded to fp32 HERE, so the
    double oracle and the fp32 library read the very same real numbers.
  * mesh edges are plain doubles (the traversal is fp64 on both sides).
  * ray record (AoS, 8 fields): x, y, z, u, v, w, E, W.

No interpolation, traversal or scoring arithmetic lives in this file.
"""
from __future__ import annotations

from dataclasses import dataclass, field
from typing import List, Tuple

import numpy as np

BASE_SEED = 1706074760

CONFIG_NAMES = {
    1: "tiny_slab_10x10x10",
    2: "criticality_like_200x200x100",
    3: "pwr17x17_like_170x170x300",
    4: "stress_512x512x512",
    5: "contention_64x64x64",
}

# rays per batch at BASELINE.json's full size (config 4: 100 such batches)
FULL_RAYS = {1: 10_000, 2: 1_000_000, 3: 10_000_000, 4: 1_000_000, 5: 10_000_000}

# (density g/cc, potential term p, 1/v coefficient a) -- SURVEY.md §8(d)
MATERIALS = {
    "air": (0.0012, 0.10, 0.01),
    "concrete": (2.3, 0.08, 0.01),
    "fissile_solution": (1.6, 0.25, 0.5),
    "uo2": (10.4, 0.02, 0.05),
    "zircaloy": (6.55, 0.04, 0.002),
    "b4c": (1.8, 0.10, 20.0),
    "borated_water": (0.74, 0.30, 0.05),
}

E_LO, E_HI = 1.0e-11, 20.0  # MeV, span of every energy grid


def rng_for(config: int, stream: int, batch: int = 0) -> np.random.Generator:
    return np.random.Generator(
        np.random.PCG64(np.random.SeedSequence([BASE_SEED, config, stream, batch]))
    )


_ROUND_FP32 = True  # False only inside make_problem(..., double_inputs=True)


def f32r(a) -> np.ndarray:
    """Round to the nearest fp32 value, return as float64 (reading Q2).  Inside make_problem(double_inputs=True)
    nothing is rounded: the all-double mode is then fed values that are NOT fp32-representable."""
    a = np.asarray(a, dtype=np.float64)
    return a.astype(np.float32).astype(np.float64) if _ROUND_FP32 else a.copy()


@dataclass
class Problem:
    config: int
    name: str
    nx: int
    ny: int
    nz: int
    xe: np.ndarray  # float64 [nx+1]
    ye: np.ndarray
    ze: np.ndarray
    material_names: List[str]
    density: np.ndarray  # float64 [M], fp32-representable
    K: int
    cell_mat: np.ndarray  # int32 [ncell, K], -1 = empty slot; cell c = ix + nx*(iy + ny*iz)
    cell_frac: np.ndarray  # float64 [ncell, K], fp32-representable
    xs: List[Tuple[np.ndarray, np.ndarray]] = field(default_factory=list)  # (E, sigma) per material

    @property
    def M(self) -> int:
        return len(self.density)

    @property
    def ncell(self) -> int:
        return self.nx * self.ny * self.nz


# --------------------------------------------------------------------------- tables
def energy_grid(n: int) -> np.ndarray:
    k = np.arange(n, dtype=np.float64)
    e = f32r(E_LO * (E_HI / E_LO) ** (k / (n - 1)))
    e[0], e[-1] = f32r(E_LO), f32r(E_HI)
    assert np.all(np.diff(e) > 0), "energy grid must stay strictly increasing after fp32 rounding"
    return e


def xs_table(config: int, stream: int, n: int, p: float, a: float, n_res: int):
    """sigma(E) = p + a*sqrt(2.53e-8/E) + sum_r H_r exp(-((lnE - lnE_r)/w_r)^2 / 2), cm^2/g."""
    g = rng_for(config, stream)
    e = energy_grid(n)
    ln_e = np.log(e)
    delta = np.log(E_HI / E_LO) / (n - 1)
    sig = p + a * np.sqrt(2.53e-8 / e)
    ln_er = np.log(1e-6) + g.random(n_res) * np.log(1e-1 / 1e-6)
    h = p * 10.0 ** (2.5 * g.random(n_res))
    w = 5.0 * delta * 10.0 ** g.random(n_res)  # log-uniform in 5..50 grid spacings
    for r in range(n_res):
        # a resonance is negligible (exp(-50)) beyond 10 widths: add it on that window only
        lo = np.searchsorted(ln_e, ln_er[r] - 10.0 * w[r])
        hi = np.searchsorted(ln_e, ln_er[r] + 10.0 * w[r])
        z = (ln_e[lo:hi] - ln_er[r]) / w[r]
        sig[lo:hi] += h[r] * np.exp(-0.5 * z * z)
    return e, f32r(sig)


def _tables(config: int, names: List[str], n: int, n_res: int):
    return [xs_table(config, 1 + m, n, MATERIALS[nm][1], MATERIALS[nm][2], n_res) for m, nm in enumerate(names)]


def _densities(names: List[str]) -> np.ndarray:
    return f32r([MATERIALS[nm][0] for nm in names])


# --------------------------------------------------------------------------- config 1
def config1(n_e: int = 1000) -> Problem:
    nx = ny = nz = 10
    names = ["air", "concrete"]
    iz = np.arange(nz)
    mat_z = np.where(iz < 3, 1, 0).astype(np.int32)  # concrete where z < 3 cm
    cell_mat = np.broadcast_to(mat_z[:, None, None], (nz, ny, nx)).reshape(-1, 1).copy()
    cell_frac = np.ones((nx * ny * nz, 1))
    ed = np.arange(nx + 1, dtype=np.float64)
    return Problem(1, CONFIG_NAMES[1], nx, ny, nz, ed.copy(), ed.copy(), ed.copy(), names, _densities(names),
                   1, cell_mat, cell_frac, _tables(1, names, n_e, 5))


# --------------------------------------------------------------------------- config 2
def config2(nx: int = 200, ny: int = 200, nz: int = 100, n_e: int = 20_000) -> Problem:
    h = 10.0
    names = ["air", "concrete", "fissile_solution"]
    ix = np.arange(nx)[None, None, :]
    iy = np.arange(ny)[None, :, None]
    iz = np.arange(nz)[:, None, None]
    wall = (iz < 3) | (ix < 3) | (ix >= nx - 3) | (iy < 3) | (iy >= ny - 3)  # floor + 4 side walls, no ceiling
    cube = (ix >= 13) & (ix < 23) & (iy >= 13) & (iy < 23) & (iz >= 3) & (iz < 13)
    mat = np.zeros((nz, ny, nx), dtype=np.int32)
    mat[np.broadcast_to(wall, mat.shape)] = 1
    mat[np.broadcast_to(cube, mat.shape)] = 2
    return Problem(2, CONFIG_NAMES[2], nx, ny, nz, h * np.arange(nx + 1), h * np.arange(ny + 1), h * np.arange(nz + 1),
                   names, _densities(names), 1, mat.reshape(-1, 1), np.ones((nx * ny * nz, 1)),
                   _tables(2, names, n_e, 50))


# --------------------------------------------------------------------------- config 3
PWR_SIDE = 21.5
PWR_HEIGHT = 365.76
PWR_PITCH = PWR_SIDE / 17
PWR_R_PELLET = 0.41
PWR_R_CLAD = 0.475


def pwr_sites():
    """17x17 site kinds: 0 fuel, 1 guide tube with B4C rod, 2 water (centre)."""
    kind = np.zeros((17, 17), dtype=np.int32)
    gt = [(r, c) for r in (2, 14) for c in (5, 8, 11)]
    gt += [(r, c) for r in (3, 13) for c in (3, 13)]
    gt += [(r, c) for r in (5, 11) for c in (2, 5, 8, 11, 14)]
    gt += [(8, c) for c in (2, 5, 11, 14)]
    assert len(gt) == 24
    for r, c in gt:
        kind[r, c] = 1
    kind[8, 8] = 2
    assert int((kind == 0).sum()) == 264
    return kind


def config3(nx: int = 170, ny: int = 170, nz: int = 300, n_e: int = 50_000, sub: int = 16) -> Problem:
    names = ["uo2", "zircaloy", "b4c", "borated_water"]
    kind = pwr_sites()
    xe = np.arange(nx + 1) * (PWR_SIDE / nx)
    ye = np.arange(ny + 1) * (PWR_SIDE / ny)
    ze = np.arange(nz + 1) * (PWR_HEIGHT / nz)
    # material of each xy sub-sample point (sub x sub per cell), z-invariant
    sx = (np.arange(nx * sub) + 0.5) * (PWR_SIDE / (nx * sub))
    sy = (np.arange(ny * sub) + 0.5) * (PWR_SIDE / (ny * sub))
    col = np.minimum((sx / PWR_PITCH).astype(np.int64), 16)
    row = np.minimum((sy / PWR_PITCH).astype(np.int64), 16)
    dx = sx - (col + 0.5) * PWR_PITCH
    dy = sy - (row + 0.5) * PWR_PITCH
    r2 = dy[:, None] ** 2 + dx[None, :] ** 2
    k2 = kind[row[:, None], col[None, :]]
    inner = np.where(k2 == 0, 0, 2)  # uo2 pellet or b4c rod
    pmat = np.where(r2 < PWR_R_PELLET**2, inner, np.where(r2 < PWR_R_CLAD**2, 1, 3))
    pmat = np.where(k2 == 2, 3, pmat).astype(np.int32)
    M = len(names)
    counts = np.zeros((ny, nx, M))
    blk = pmat.reshape(ny, sub, nx, sub)
    for m in range(M):
        counts[:, :, m] = (blk == m).sum(axis=(1, 3))
    K = 3
    order = np.argsort(-counts, axis=2, kind="stable")[:, :, :K]  # 3 largest, ties by material id
    top = np.take_along_axis(counts, order, axis=2)
    frac = top / top.sum(axis=2, keepdims=True)
    ids = np.where(top > 0, order, -1).astype(np.int32)
    frac = f32r(np.where(top > 0, frac, 0.0))
    cell_mat = np.broadcast_to(ids[None], (nz, ny, nx, K)).reshape(-1, K).copy()
    cell_frac = np.broadcast_to(frac[None], (nz, ny, nx, K)).reshape(-1, K).copy()
    return Problem(3, CONFIG_NAMES[3], nx, ny, nz, xe, ye, ze, names, _densities(names), K, cell_mat, cell_frac,
                   _tables(3, names, n_e, 200))


# --------------------------------------------------------------------------- config 4
def config4(n: int = 512, block: int = 8, n_e: int = 100_000) -> Problem:
    names = ["air", "borated_water", "concrete", "zircaloy", "uo2"]  # densities {0.0012,0.74,2.3,6.55,10.4}
    g = rng_for(4, 0)
    nb = n // block
    assert nb * block == n
    B = nb**3
    K, M = 4, len(names)
    n_mat = 1 + np.minimum((g.random(B) * 4).astype(np.int64), 3)  # 1..4 materials in the block
    perm = np.argsort(g.random((B, M)), axis=1, kind="stable")[:, :K]  # distinct materials
    expo = -np.log(1.0 - g.random((B, K)))  # Dirichlet(1) = normalised exponentials
    live = np.arange(K)[None, :] < n_mat[:, None]
    expo = np.where(live, expo, 0.0)
    frac = f32r(expo / expo.sum(axis=1, keepdims=True))
    ids = np.where(live, perm, -1).astype(np.int32)

    def expand(a):
        a = a.reshape(nb, nb, nb, K)
        for ax in range(3):
            a = np.repeat(a, block, axis=ax)
        return a.reshape(-1, K)

    ed = np.arange(n + 1, dtype=np.float64)
    return Problem(4, CONFIG_NAMES[4] if n == 512 else f"stress_{n}^3", n, n, n, ed.copy(), ed.copy(), ed.copy(),
                   names, _densities(names), K, expand(ids), expand(frac), _tables(4, names, n_e, 500))


# --------------------------------------------------------------------------- config 5
def config5(n: int = 64, n_e: int = 200_000, n_res: int = 2000) -> Problem:
    g = rng_for(5, 0)
    M = K = 8
    names = [f"mix{m}" for m in range(M)]
    density = f32r(0.01 * 1000.0 ** g.random(M))  # log-uniform 0.01..10 g/cc
    p = 0.02 * 15.0 ** g.random(M)
    a = 0.002 * 1000.0 ** g.random(M)
    ncell = n**3
    expo = -np.log(1.0 - g.random((ncell, K)))
    frac = f32r(expo / expo.sum(axis=1, keepdims=True))
    ids = np.broadcast_to(np.arange(K, dtype=np.int32)[None, :], (ncell, K)).copy()
    ed = np.arange(n + 1, dtype=np.float64)
    xs = [xs_table(5, 1 + m, n_e, float(p[m]), float(a[m]), n_res) for m in range(M)]
    return Problem(5, CONFIG_NAMES[5], n, n, n, ed.copy(), ed.copy(), ed.copy(), names, density, K, ids, frac, xs)


def make_problem(config: int, double_inputs: bool = False, **kw) -> Problem:
    """double_inputs=True: tables, densities and fractions keep their full double values (inputs for the all-double
    mode only; the mixed library would round them and no longer read the oracle's numbers)."""
    global _ROUND_FP32
    _ROUND_FP32 = not double_inputs
    try:
        return {1: config1, 2: config2, 3: config3, 4: config4, 5: config5}[config](**kw)
    finally:
        _ROUND_FP32 = True


# --------------------------------------------------------------------------- rays
def _isotropic(g: np.random.Generator, n: int) -> np.ndarray:
    mu = 2.0 * g.random(n) - 1.0
    phi = 2.0 * np.pi * g.random(n)
    s = np.sqrt(np.maximum(0.0, 1.0 - mu * mu))
    d = np.stack([s * np.cos(phi), s * np.sin(phi), mu], axis=1)
    return d / np.linalg.norm(d, axis=1, keepdims=True)  # normalised in double, rounded to fp32 later


def _log_uniform(g, n, lo, hi):
    return lo * (hi / lo) ** g.random(n)


def _watt(g, n, a=0.988, b=2.249):
    """Watt fission spectrum ~ exp(-E/a) sinh(sqrt(bE)) by the standard Maxwellian-shift sampling."""
    x1, x2, x3, x4 = (1.0 - g.random(n) for _ in range(4))
    w = a * (-np.log(x1) - np.log(x2) * np.cos(0.5 * np.pi * x3) ** 2)
    e = w + 0.25 * a * a * b + (2.0 * x4 - 1.0) * np.sqrt(a * a * b * w)
    return np.clip(e, E_LO, E_HI)


def _pack(pos, d, e, w, lo, hi, dtype=np.float32) -> np.ndarray:
    """Round to `dtype` (fp32: the mixed-mode record; fp64: nothing is rounded) and keep origins inside the
    half-open box [lo, hi) after rounding."""
    ft = np.dtype(dtype).type
    rays = np.empty((len(e), 8), dtype=dtype)
    rays[:, 0:3] = pos
    for a in range(3):
        hi_t = np.nextafter(ft(hi[a]), ft(-np.inf)) if ft(hi[a]) >= hi[a] else ft(hi[a])
        lo_t = np.nextafter(ft(lo[a]), ft(np.inf)) if ft(lo[a]) < lo[a] else ft(lo[a])
        rays[:, a] = np.clip(rays[:, a], lo_t, hi_t)
    rays[:, 3:6] = d
    rays[:, 6] = e
    rays[:, 6] = np.clip(rays[:, 6], ft(E_LO), ft(E_HI))
    rays[:, 7] = w
    return rays


def make_rays(prob: Problem, n: int, batch: int = 0, dtype=np.float32) -> np.ndarray:
    """[n, 8] ray records for problem `prob` (shape rules per config): float32 (the mixed-mode
    record, reading Q2) or, for the all-double mode, float64 with nothing rounded."""
    c = prob.config
    g = rng_for(c, 9, batch)
    lo = (prob.xe[0], prob.ye[0], prob.ze[0])
    hi = (prob.xe[-1], prob.ye[-1], prob.ze[-1])
    span = np.array(hi) - np.array(lo)
    if c == 1:
        pos = np.array(lo) + g.random((n, 3)) * span
        e = _log_uniform(g, n, E_LO, E_HI)
    elif c == 2:
        hx, hy, hz = prob.xe[1] - prob.xe[0], prob.ye[1] - prob.ye[0], prob.ze[1] - prob.ze[0]
        c_lo = np.array([13 * hx, 13 * hy, 3 * hz])
        c_hi = np.array([23 * hx, 23 * hy, 13 * hz])
        a_lo = np.array([3 * hx, 3 * hy, 3 * hz])
        a_hi = np.array([hi[0] - 3 * hx, hi[1] - 3 * hy, hi[2]])
        in_cube = g.random(n) < 0.9
        pos = c_lo + g.random((n, 3)) * (c_hi - c_lo)
        need = np.flatnonzero(~in_cube)
        while len(need):  # rejection: uniform in the air volume (interior minus the source cube)
            cand = a_lo + g.random((len(need), 3)) * (a_hi - a_lo)
            ok = ~np.all((cand >= c_lo) & (cand < c_hi), axis=1)
            pos[need[ok]] = cand[ok]
            need = need[~ok]
        e = _watt(g, n)
    elif c == 3:
        kind = pwr_sites()
        fr, fc = np.nonzero(kind == 0)
        pin = np.minimum((g.random(n) * len(fr)).astype(np.int64), len(fr) - 1)
        rad = PWR_R_PELLET * np.sqrt(g.random(n))
        ang = 2.0 * np.pi * g.random(n)
        pos = np.stack([(fc[pin] + 0.5) * PWR_PITCH + rad * np.cos(ang),
                        (fr[pin] + 0.5) * PWR_PITCH + rad * np.sin(ang),
                        lo[2] + g.random(n) * span[2]], axis=1)
        e = _watt(g, n)
    elif c == 4:
        pos = np.array(lo) + g.random((n, 3)) * span
        e = _log_uniform(g, n, 1.0e-9, E_HI)
    elif c == 5:
        h = np.array([prob.xe[1] - prob.xe[0], prob.ye[1] - prob.ye[0], prob.ze[1] - prob.ze[0]])
        first = np.array([prob.nx, prob.ny, prob.nz]) // 2 - 2  # cells [30,34)^3 at n = 64
        pos = np.array(lo) + (first + 4.0 * g.random((n, 3))) * h
        e = _log_uniform(g, n, E_LO, E_HI)
    else:
        raise ValueError(c)
    d = _isotropic(g, n)
    w = 0.5 + g.random(n)
    return _pack(pos, d, e, w, lo, hi, dtype)


# --------------------------------------------------------------------------- multi-nuclide materials (NEXT-4)
def add_nuclides(prob, n_nuclides: int = 6, max_per_material: int = 4, keep_direct: int = 1, seed_stream: int = 20):
    """Returns a shallow copy of `prob` in which every material but the first `keep_direct` is a mixture of
    nuclides: sigma_m(E) = sum_j w_j sigma_nuclide_j(E).  Nuclide tables are synthetic (same recipe as the
    material tables) on grids of DIFFERENT sizes (no unionised grid), weights are fp32-representable mass
    fractions that sum to about 1.  Input generation only: no method arithmetic."""
    import copy

    g = rng_for(prob.config, seed_stream)
    q = copy.copy(prob)
    n_e = max(len(e) for e, _ in prob.xs)
    sizes = [max(9, int(n_e * f)) for f in (1.0, 0.5, 0.37, 0.81, 0.25, 0.66, 0.45, 0.9)]
    q.nuclide_xs = [xs_table(prob.config, seed_stream + 1 + j, sizes[j % len(sizes)], 0.05 + 0.3 * g.random(),
                             0.01 * 10.0 ** (2.0 * g.random()), max(3, min(200, sizes[j % len(sizes)] // 200)))
                    for j in range(n_nuclides)]
    q.mixtures = []
    q.xs = list(prob.xs)
    for m in range(prob.M):
        if m < keep_direct:
            q.mixtures.append(None)
            continue
        k = int(g.integers(1, max_per_material + 1))
        ids = g.choice(n_nuclides, size=min(k, n_nuclides), replace=False).astype(np.int32)
        w = g.random(len(ids)) + 0.05
        q.mixtures.append((ids, f32r(w / w.sum())))
        q.xs[m] = None
    return q


# --------------------------------------------------------------------------- R-Z pin-cell-like problem (NEXT-4)
def make_rz_problem(nr: int = 256, nz: int = 512, n_e: int = 20_000, double_inputs: bool = False):
    global _ROUND_FP32
    _ROUND_FP32 = not double_inputs
    try:
        return _make_rz_problem(nr, nz, n_e)
    finally:
        _ROUND_FP32 = True


def _make_rz_problem(nr: int, nz: int, n_e: int):
    """One fuel-pin cell seen as an R-Z mesh: UO2 to r = 0.41 cm, zircaloy to 0.475 cm, borated water out to the
    equivalent-cell radius 0.7135 cm (pitch/sqrt(pi)), 365.76 cm high; nr equal shells, nz equal slabs, K = 1.
    Stands in for the paper's wish for 2-D cylindrical meshes; inputs only."""
    from types import SimpleNamespace

    names = ["uo2", "zircaloy", "borated_water"]
    r_out = PWR_PITCH / np.sqrt(np.pi)
    re = r_out * np.arange(nr + 1) / nr
    ze = PWR_HEIGHT * np.arange(nz + 1) / nz
    rc = 0.5 * (re[1:] + re[:-1])
    shell_mat = np.where(rc < PWR_R_PELLET, 0, np.where(rc < PWR_R_CLAD, 1, 2)).astype(np.int32)
    cell_mat = np.tile(shell_mat, nz).reshape(-1, 1)
    return SimpleNamespace(config=3, name=f"rz_pin_cell_{nr}x{nz}", nx=nr, ny=1, nz=nz, nr=nr, re=re, ze=ze, xe=re,
                           ye=np.array([0.0, 1.0]), density=_densities(names), K=1, cell_mat=cell_mat,
                           cell_frac=np.ones((nr * nz, 1)), xs=_tables(3, names, n_e, 50), M=3, ncell=nr * nz,
                           material_names=names)


def make_rz_rays(prob, n: int, batch: int = 0, dtype=np.float32) -> np.ndarray:
    """Rays born uniformly in the fuel (rho < 0.41 cm), isotropic, Watt energies; [n, 8] float32 (or float64, unrounded)."""
    g = rng_for(3, 11, batch)
    rho = PWR_R_PELLET * np.sqrt(g.random(n))
    phi = 2.0 * np.pi * g.random(n)
    z = prob.ze[0] + g.random(n) * (prob.ze[-1] - prob.ze[0])
    pos = np.stack([rho * np.cos(phi), rho * np.sin(phi), z], axis=1)
    d = _isotropic(g, n)
    ft = np.dtype(dtype).type
    rays = np.concatenate([pos, d, _watt(g, n)[:, None], (0.5 + g.random(n))[:, None]], axis=1).astype(dtype)
    rays[:, 2] = np.clip(rays[:, 2], ft(prob.ze[0]), np.nextafter(ft(prob.ze[-1]), ft(0)))
    return np.ascontiguousarray(rays)
