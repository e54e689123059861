"""Tiny random problems for pins and property tests (input generation only; no method arithmetic)."""
from __future__ import annotations

from types import SimpleNamespace

import numpy as np


def f32r(a):
    return np.asarray(a, dtype=np.float64).astype(np.float32).astype(np.float64)


def tiny_problem(seed, nx=4, ny=3, nz=5, M=3, K=2, n_e=17, uniform=False, void=False, homogeneous=False,
                 fp32_values=True):
    g = np.random.default_rng(seed)
    rnd = f32r if fp32_values else (lambda a: np.asarray(a, dtype=np.float64))

    def edges(n):
        if uniform:
            return -1.0 + 0.75 * np.arange(n + 1)
        return np.concatenate([[-1.0], -1.0 + np.cumsum(0.2 + g.random(n))])

    xe, ye, ze = edges(nx), edges(ny), edges(nz)
    ncell = nx * ny * nz
    density = rnd(0.5 + 3.0 * g.random(M))
    if void:
        density = np.zeros(M)
    cell_mat = g.integers(-1, M, size=(ncell, K)).astype(np.int32)
    cell_frac = rnd(g.random((ncell, K)))
    cell_frac[cell_mat < 0] = 0.0
    if homogeneous:
        cell_mat[:] = -1
        cell_mat[:, 0] = 0
        cell_frac[:] = 0.0
        cell_frac[:, 0] = 1.0
    xs = []
    for m in range(M):
        e = rnd(np.sort(1e-3 * 1e4 ** g.random(n_e)))
        e = np.unique(e)
        s = rnd(0.05 + g.random(len(e)))
        xs.append((e, s))
    return SimpleNamespace(config=0, name=f"tiny{seed}", nx=nx, ny=ny, nz=nz, xe=xe, ye=ye, ze=ze,
                           density=density, K=K, cell_mat=cell_mat, cell_frac=cell_frac, xs=xs,
                           M=M, ncell=ncell)


def tiny_rays(prob, seed, n, axis_aligned_share=0.0, e_lo=5e-4, e_hi=20.0, dtype=np.float32):
    g = np.random.default_rng(seed)
    lo = np.array([prob.xe[0], prob.ye[0], prob.ze[0]])
    hi = np.array([prob.xe[-1], prob.ye[-1], prob.ze[-1]])
    pos = lo + (0.001 + 0.998 * g.random((n, 3))) * (hi - lo)
    d = g.normal(size=(n, 3))
    d /= np.linalg.norm(d, axis=1, keepdims=True)
    k = int(axis_aligned_share * n)
    for r in range(k):  # zero out one or two components (exercises Q10, including -0.0)
        z = g.permutation(3)[: 1 + (r % 2)]
        d[r, z] = 0.0 if r % 3 else -0.0
        d[r] /= np.linalg.norm(d[r])
    e = e_lo * (e_hi / e_lo) ** g.random(n)
    w = 0.5 + g.random(n)
    rays = np.concatenate([pos, d, e[:, None], w[:, None]], axis=1)
    return np.ascontiguousarray(rays.astype(dtype))


def tiny_rz_problem(seed, nr=5, nz=4, M=3, K=2, n_e=17, uniform=False, void=False, homogeneous=False, fp32_values=True):
    """A tiny R-Z problem: tiny_problem's materials and tables on nr radial shells (from r = 0) x nz axial slabs.
    Returned with nx = nr, ny = 1 (cell c = ir + nr*iz) and the extra fields re, ze, nr."""
    prob = tiny_problem(seed, nx=nr, ny=1, nz=nz, M=M, K=K, n_e=n_e, uniform=uniform, void=void, homogeneous=homogeneous,
                        fp32_values=fp32_values)
    g = np.random.default_rng(seed + 1000)
    prob.re = 0.5 * np.arange(nr + 1) if uniform else np.concatenate([[0.0], np.cumsum(0.15 + 0.6 * g.random(nr))])
    prob.nr = nr
    prob.xe, prob.ye = prob.re, np.array([0.0, 1.0])
    return prob


def tiny_rz_rays(prob, seed, n, axis_parallel_share=0.0, through_axis_share=0.0, e_lo=5e-4, e_hi=20.0, dtype=np.float32):
    g = np.random.default_rng(seed)
    R = prob.re[-1]
    rho = R * np.sqrt(0.999 * g.random(n))
    phi = 2 * np.pi * g.random(n)
    z = prob.ze[0] + (0.001 + 0.998 * g.random(n)) * (prob.ze[-1] - prob.ze[0])
    pos = np.stack([rho * np.cos(phi), rho * np.sin(phi), z], axis=1)
    d = g.normal(size=(n, 3))
    d /= np.linalg.norm(d, axis=1, keepdims=True)
    k = int(axis_parallel_share * n)
    d[:k, :2] = 0.0
    d[:k, 2] = np.where(g.random(k) < 0.5, -1.0, 1.0)
    j = int(through_axis_share * n)
    for r in range(k, k + j):      # aimed exactly at the axis in the xy plane (in fp32 inputs: nearly)
        s = -pos[r, :2] / max(np.linalg.norm(pos[r, :2]), 1e-30)
        d[r, :2] = s * np.linalg.norm(d[r, :2])
    e = e_lo * (e_hi / e_lo) ** g.random(n)
    w = 0.5 + g.random(n)
    rays = np.concatenate([pos, d, e[:, None], w[:, None]], axis=1)
    return np.ascontiguousarray(rays.astype(dtype))


def tiny_sphere_problem(seed, nr=6, M=3, K=2, n_e=17, uniform=False, homogeneous=False, fp32_values=True):
    """Tiny 1-D spherical problem: nr shells about the origin (cell c = ir); fields re, nr, sphere=True."""
    prob = tiny_problem(seed, nx=nr, ny=1, nz=1, M=M, K=K, n_e=n_e, uniform=uniform, homogeneous=homogeneous,
                        fp32_values=fp32_values)
    g = np.random.default_rng(seed + 2000)
    prob.re = 0.5 * np.arange(nr + 1) if uniform else np.concatenate([[0.0], np.cumsum(0.15 + 0.6 * g.random(nr))])
    prob.nr = nr
    prob.sphere = True
    prob.xe, prob.ye, prob.ze = prob.re, np.array([0.0, 1.0]), np.array([0.0, 1.0])
    return prob


def tiny_sphere_rays(prob, seed, n, through_centre_share=0.0, e_lo=5e-4, e_hi=20.0, dtype=np.float32):
    g = np.random.default_rng(seed)
    R = prob.re[-1]
    u = g.normal(size=(n, 3))
    u /= np.linalg.norm(u, axis=1, keepdims=True)
    pos = u * (R * np.cbrt(0.999 * g.random(n)))[:, None]
    d = g.normal(size=(n, 3))
    d /= np.linalg.norm(d, axis=1, keepdims=True)
    k = int(through_centre_share * n)
    d[:k] = -pos[:k] / np.maximum(np.linalg.norm(pos[:k], axis=1, keepdims=True), 1e-30)
    e = e_lo * (e_hi / e_lo) ** g.random(n)
    w = 0.5 + g.random(n)
    rays = np.concatenate([pos, d, e[:, None], w[:, None]], axis=1)
    return np.ascontiguousarray(rays.astype(dtype))
