"""ctypes loader for the CPU oracle (oracle/vrc_oracle.c).

TEST INFRASTRUCTURE, NOT THE PRODUCT: only tests/, __graft_entry__.smoke() and
bench.py's cpu_baseline / --impl reference legs may import this module.  It does not
import, and is not imported by, anything under paper_1706_07476_b200/.

The shared object is built on first use with
    gcc -O2 -ffp-contract=off -fopenmp -shared -fPIC vrc_oracle.c -lm
(no fast-math, no FMA contraction -- see the header of vrc_oracle.c).
"""
from __future__ import annotations

import ctypes as C
import os
import subprocess
from dataclasses import dataclass
from typing import Optional

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "vrc_oracle.c")
_LIB = os.path.join(_HERE, "libvrc_oracle.so")
_lib = None


def build(force: bool = False) -> str:
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        tmp = _LIB + f".{os.getpid()}.tmp"
        subprocess.check_call(["gcc", "-O2", "-ffp-contract=off", "-fopenmp", "-shared", "-fPIC",
                               "-o", tmp, _SRC, "-lm"])
        os.replace(tmp, _LIB)
    return _LIB


class _Problem(C.Structure):
    _fields_ = [("nx", C.c_int32), ("ny", C.c_int32), ("nz", C.c_int32),
                ("xe", C.c_void_p), ("ye", C.c_void_p), ("ze", C.c_void_p),
                ("M", C.c_int32), ("density", C.c_void_p), ("K", C.c_int32),
                ("cell_mat", C.c_void_p), ("cell_frac", C.c_void_p),
                ("xs_off", C.c_void_p), ("xs_E", C.c_void_p), ("xs_sig", C.c_void_p),
                ("N", C.c_int32), ("nxs_off", C.c_void_p), ("nxs_E", C.c_void_p), ("nxs_sig", C.c_void_p),
                ("mix_off", C.c_void_p), ("mix_nuc", C.c_void_p), ("mix_w", C.c_void_p)]


class _Counts(C.Structure):
    _fields_ = [("rays_accepted", C.c_int64), ("rays_rejected", C.c_int64), ("segments", C.c_int64)]


class _RzMesh(C.Structure):
    _fields_ = [("nr", C.c_int32), ("nz", C.c_int32), ("re", C.c_void_p), ("ze", C.c_void_p), ("spherical", C.c_int32)]


class _NeDiag(C.Structure):
    _fields_ = [("nseg", C.c_void_p), ("hash", C.c_void_p), ("tau", C.c_void_p), ("score", C.c_void_p)]


class _Diag(C.Structure):
    _fields_ = [("nseg", C.c_void_p), ("hash", C.c_void_p), ("sum_l", C.c_void_p), ("t_exit", C.c_void_p),
                ("tau_exit", C.c_void_p), ("sum_score", C.c_void_p), ("sum_sig_score", C.c_void_p),
                ("cells", C.c_void_p), ("lens", C.c_void_p), ("scores", C.c_void_p), ("cap", C.c_int64)]


def _load():
    global _lib
    if _lib is None:
        _lib = C.CDLL(build())
        _lib.vrc_sigma.restype = C.c_double
        _lib.vrc_sigma.argtypes = [C.POINTER(_Problem), C.c_int32, C.c_double]
        _lib.vrc_cast.restype = C.c_int
        _lib.vrc_cast.argtypes = [C.POINTER(_Problem), C.c_int64, C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p]
        _lib.vrc_cast_mt.restype = C.c_int
        _lib.vrc_cast_mt.argtypes = [C.POINTER(_Problem), C.c_int64, C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p,
                                     C.c_int, C.c_int64]
        _lib.vrc_next_event.restype = C.c_int
        _lib.vrc_next_event.argtypes = [C.POINTER(_Problem), C.c_int64, C.c_void_p, C.c_void_p, C.c_void_p,
                                        C.c_void_p, C.c_void_p]
        _lib.vrc_cast_rz.restype = C.c_int
        _lib.vrc_cast_rz.argtypes = [C.POINTER(_Problem), C.POINTER(_RzMesh), C.c_int64, C.c_void_p, C.c_void_p,
                                     C.c_void_p, C.c_void_p]
        _lib.vrc_next_event_rz.restype = C.c_int
        _lib.vrc_next_event_rz.argtypes = [C.POINTER(_Problem), C.POINTER(_RzMesh), C.c_int64, C.c_void_p, C.c_void_p,
                                           C.c_void_p, C.c_void_p, C.c_void_p]
        _lib.vrc_fnv1a_cells.restype = C.c_uint64
        _lib.vrc_fnv1a_cells.argtypes = [C.c_void_p, C.c_int64]
        _lib.vrc_max_threads.restype = C.c_int
    return _lib


def fnv1a_cells(cells) -> int:
    a = np.ascontiguousarray(cells, dtype=np.uint32)
    return int(_load().vrc_fnv1a_cells(a.ctypes.data, a.size))


def max_threads() -> int:
    return int(_load().vrc_max_threads())


@dataclass
class CastResult:
    tally: Optional[np.ndarray]
    rays_accepted: int
    rays_rejected: int
    segments: int
    threads: int
    nseg: Optional[np.ndarray] = None
    hash: Optional[np.ndarray] = None
    sum_l: Optional[np.ndarray] = None
    t_exit: Optional[np.ndarray] = None
    tau_exit: Optional[np.ndarray] = None
    sum_score: Optional[np.ndarray] = None
    sum_sig_score: Optional[np.ndarray] = None
    cells: Optional[np.ndarray] = None
    lens: Optional[np.ndarray] = None
    scores: Optional[np.ndarray] = None


@dataclass
class NextEventResult:
    det_sum: float
    rays_accepted: int
    rays_rejected: int
    segments: int
    nseg: np.ndarray
    hash: np.ndarray
    tau: np.ndarray
    score: np.ndarray


class Oracle:
    """The oracle bound to one problem (mesh + materials + tables).

    `prob` is any object with nx, ny, nz, xe, ye, ze, density, K, cell_mat, cell_frac, xs
    (e.g. workloads.Problem).  Arrays are taken as float64 / int32 views, never modified.
    """

    def __init__(self, prob):
        self.lib = _load()
        self.nx, self.ny, self.nz = int(prob.nx), int(prob.ny), int(prob.nz)
        self.ncell = self.nx * self.ny * self.nz
        self._xe = np.ascontiguousarray(prob.xe, dtype=np.float64)
        self._ye = np.ascontiguousarray(prob.ye, dtype=np.float64)
        self._ze = np.ascontiguousarray(prob.ze, dtype=np.float64)
        self._den = np.ascontiguousarray(prob.density, dtype=np.float64)
        self.M = len(self._den)
        self.K = int(prob.K)
        self._mat = np.ascontiguousarray(prob.cell_mat, dtype=np.int32).reshape(-1)
        self._frac = np.ascontiguousarray(prob.cell_frac, dtype=np.float64).reshape(-1)
        assert self._mat.size == self.ncell * self.K and self._frac.size == self.ncell * self.K
        assert len(prob.xs) == self.M and self.M <= 64
        # optional multi-nuclide materials: prob.nuclide_xs = [(E, sigma)], prob.mixtures[m] = (nuclide ids, weights) | None
        mixtures = getattr(prob, "mixtures", None) or [None] * self.M
        nuclide_xs = getattr(prob, "nuclide_xs", None) or []
        off = np.zeros(self.M + 1, dtype=np.int64)
        tabs = []
        for m, t in enumerate(prob.xs):
            if mixtures[m] is not None:
                off[m + 1] = off[m]          # no table of its own
                continue
            e, s = t
            assert len(e) == len(s) and len(e) >= 1
            off[m + 1] = off[m] + len(e)
            tabs.append((e, s))
        self._off = off
        self._E = np.ascontiguousarray(np.concatenate([np.asarray(e, dtype=np.float64) for e, _ in tabs] or [np.zeros(1)]))
        self._S = np.ascontiguousarray(np.concatenate([np.asarray(s, dtype=np.float64) for _, s in tabs] or [np.zeros(1)]))
        self.N = len(nuclide_xs)
        noff = np.zeros(self.N + 1, dtype=np.int64)
        for q, (e, s) in enumerate(nuclide_xs):
            assert len(e) == len(s) and len(e) >= 1
            noff[q + 1] = noff[q] + len(e)
        self._noff = noff
        self._nE = np.ascontiguousarray(np.concatenate([np.asarray(e, dtype=np.float64) for e, _ in nuclide_xs] or [np.zeros(1)]))
        self._nS = np.ascontiguousarray(np.concatenate([np.asarray(s, dtype=np.float64) for _, s in nuclide_xs] or [np.zeros(1)]))
        moff = np.zeros(self.M + 1, dtype=np.int64)
        mn, mw = [], []
        for m in range(self.M):
            k = 0
            if mixtures[m] is not None:
                ids, w = mixtures[m]
                assert len(ids) == len(w) and len(ids) >= 1 and all(0 <= int(q) < self.N for q in ids)
                mn += [int(q) for q in ids]
                mw += [float(x) for x in w]
                k = len(ids)
            moff[m + 1] = moff[m] + k
        self._moff = moff
        self._mn = np.ascontiguousarray(np.array(mn or [0], dtype=np.int32))
        self._mw = np.ascontiguousarray(np.array(mw or [0.0], dtype=np.float64))
        self._p = _Problem(self.nx, self.ny, self.nz, self._xe.ctypes.data, self._ye.ctypes.data,
                           self._ze.ctypes.data, self.M, self._den.ctypes.data, self.K, self._mat.ctypes.data,
                           self._frac.ctypes.data, self._off.ctypes.data, self._E.ctypes.data, self._S.ctypes.data,
                           self.N, self._noff.ctypes.data, self._nE.ctypes.data, self._nS.ctypes.data,
                           self._moff.ctypes.data, self._mn.ctypes.data, self._mw.ctypes.data)

    def sigma(self, m: int, E: float) -> float:
        return float(self.lib.vrc_sigma(C.byref(self._p), int(m), float(E)))

    def cast(self, rays, tally: Optional[np.ndarray] = None, *, score: bool = True, per_ray: bool = False,
             cap: int = 0, threads: int = 1, private_bytes_max: int = 8 << 30) -> CastResult:
        """Cast `rays` ([n,8], any float dtype; promoted exactly to double).

        score=False walks without touching a tally (trace only).  per_ray=True returns the O6
        per-ray diagnostics; cap>0 also returns the first `cap` (cell, length, score) of each ray.
        """
        r = np.ascontiguousarray(np.asarray(rays, dtype=np.float64).reshape(-1, 8))
        n = r.shape[0]
        if score and tally is None:
            tally = np.zeros(self.ncell, dtype=np.float64)
        if tally is not None:
            assert tally.dtype == np.float64 and tally.size == self.ncell and tally.flags.c_contiguous
        res = CastResult(tally if score else None, 0, 0, 0, 1)
        dg = None
        if per_ray or cap > 0:
            res.nseg = np.zeros(n, dtype=np.uint32)
            res.hash = np.zeros(n, dtype=np.uint64)
            for nm in ("sum_l", "t_exit", "tau_exit", "sum_score", "sum_sig_score"):
                setattr(res, nm, np.zeros(n, dtype=np.float64))
            dg = _Diag(res.nseg.ctypes.data, res.hash.ctypes.data, res.sum_l.ctypes.data, res.t_exit.ctypes.data,
                       res.tau_exit.ctypes.data, res.sum_score.ctypes.data, res.sum_sig_score.ctypes.data,
                       None, None, None, 0)
            if cap > 0:
                res.cells = np.full((n, cap), -1, dtype=np.int32)
                res.lens = np.zeros((n, cap), dtype=np.float64)
                res.scores = np.zeros((n, cap), dtype=np.float64)
                dg.cells, dg.lens, dg.scores, dg.cap = res.cells.ctypes.data, res.lens.ctypes.data, res.scores.ctypes.data, cap
        cnt = _Counts()
        tptr = tally.ctypes.data if (score and tally is not None) else None
        dptr = C.cast(C.byref(dg), C.c_void_p) if dg is not None else None
        if threads <= 1:
            rc = self.lib.vrc_cast(C.byref(self._p), n, r.ctypes.data, tptr, dptr, C.cast(C.byref(cnt), C.c_void_p))
            used = 1
        else:
            rc = self.lib.vrc_cast_mt(C.byref(self._p), n, r.ctypes.data, tptr, dptr,
                                      C.cast(C.byref(cnt), C.c_void_p), int(threads), int(private_bytes_max))
            used = rc
        if rc < 0:
            raise RuntimeError(f"oracle error {rc}")
        res.rays_accepted, res.rays_rejected, res.segments, res.threads = (
            int(cnt.rays_accepted), int(cnt.rays_rejected), int(cnt.segments), int(used))
        return res

    def cast_sphere(self, rays, re, *, cap: int = 0) -> CastResult:
        """Cast `rays` on 1-D spherical shells (re: nr+1 radii from 0 about the origin); cell c = ir."""
        return self.cast_rz(rays, re, np.array([0.0, 1.0]), cap=cap, spherical=True)

    def cast_rz(self, rays, re, ze, *, per_ray: bool = True, cap: int = 0, spherical: bool = False) -> CastResult:
        """Cast `rays` on the R-Z mesh (re: nr+1 radii from 0, ze: nz+1 planes); the problem's cell arrays hold
        nr*nz cells, c = ir + nr*iz (steps Z1..Z5 of vrc_oracle.c).  Single thread."""
        r = np.ascontiguousarray(np.asarray(rays, dtype=np.float64).reshape(-1, 8))
        n = r.shape[0]
        re = np.ascontiguousarray(re, dtype=np.float64)
        ze = np.ascontiguousarray(ze, dtype=np.float64)
        nr, nz = len(re) - 1, len(ze) - 1
        assert nr * nz == self.ncell, "the problem's cell arrays must hold nr*nz cells"
        tally = np.zeros(self.ncell, dtype=np.float64)
        res = CastResult(tally, 0, 0, 0, 1)
        res.nseg = np.zeros(n, dtype=np.uint32)
        res.hash = np.zeros(n, dtype=np.uint64)
        for nm in ("sum_l", "t_exit", "tau_exit", "sum_score", "sum_sig_score"):
            setattr(res, nm, np.zeros(n, dtype=np.float64))
        dg = _Diag(res.nseg.ctypes.data, res.hash.ctypes.data, res.sum_l.ctypes.data, res.t_exit.ctypes.data,
                   res.tau_exit.ctypes.data, res.sum_score.ctypes.data, res.sum_sig_score.ctypes.data, None, None, None, 0)
        if cap > 0:
            res.cells = np.full((n, cap), -1, dtype=np.int32)
            res.lens = np.zeros((n, cap), dtype=np.float64)
            res.scores = np.zeros((n, cap), dtype=np.float64)
            dg.cells, dg.lens, dg.scores, dg.cap = res.cells.ctypes.data, res.lens.ctypes.data, res.scores.ctypes.data, cap
        g = _RzMesh(nr, nz, re.ctypes.data, ze.ctypes.data, 1 if spherical else 0)
        cnt = _Counts()
        rc = self.lib.vrc_cast_rz(C.byref(self._p), C.byref(g), n, r.ctypes.data, tally.ctypes.data,
                                  C.cast(C.byref(dg), C.c_void_p), C.cast(C.byref(cnt), C.c_void_p))
        if rc < 0:
            raise RuntimeError(f"oracle error {rc}")
        res.rays_accepted, res.rays_rejected, res.segments = int(cnt.rays_accepted), int(cnt.rays_rejected), int(cnt.segments)
        return res

    def next_event(self, rays, det) -> NextEventResult:
        """Next-event (point-detector) estimator of `rays` ([n,8]; direction fields ignored) for ONE detector
        point `det` (x, y, z): steps N1..N6 of vrc_oracle.c.  Returns the detector sum and per-event outputs."""
        r = np.ascontiguousarray(np.asarray(rays, dtype=np.float64).reshape(-1, 8))
        n = r.shape[0]
        d = np.ascontiguousarray(np.asarray(det, dtype=np.float64).reshape(3))
        nseg = np.zeros(n, dtype=np.uint32)
        hsh = np.zeros(n, dtype=np.uint64)
        tau = np.zeros(n, dtype=np.float64)
        score = np.zeros(n, dtype=np.float64)
        dg = _NeDiag(nseg.ctypes.data, hsh.ctypes.data, tau.ctypes.data, score.ctypes.data)
        total = C.c_double(0.0)
        cnt = _Counts()
        rc = self.lib.vrc_next_event(C.byref(self._p), n, r.ctypes.data, d.ctypes.data,
                                     C.cast(C.byref(total), C.c_void_p), C.cast(C.byref(dg), C.c_void_p),
                                     C.cast(C.byref(cnt), C.c_void_p))
        if rc < 0:
            raise RuntimeError(f"oracle error {rc}")
        return NextEventResult(float(total.value), int(cnt.rays_accepted), int(cnt.rays_rejected), int(cnt.segments),
                               nseg, hsh, tau, score)


    def _next_event_rz(self, rays, det, re, ze, spherical) -> NextEventResult:
        r = np.ascontiguousarray(np.asarray(rays, dtype=np.float64).reshape(-1, 8))
        n = r.shape[0]
        d = np.ascontiguousarray(np.asarray(det, dtype=np.float64).reshape(3))
        re = np.ascontiguousarray(re, dtype=np.float64)
        ze = np.ascontiguousarray(ze, dtype=np.float64)
        nr, nz = len(re) - 1, len(ze) - 1
        assert nr * nz == self.ncell, "the problem's cell arrays must hold nr*nz cells"
        nseg = np.zeros(n, dtype=np.uint32)
        hsh = np.zeros(n, dtype=np.uint64)
        tau = np.zeros(n, dtype=np.float64)
        score = np.zeros(n, dtype=np.float64)
        dg = _NeDiag(nseg.ctypes.data, hsh.ctypes.data, tau.ctypes.data, score.ctypes.data)
        g = _RzMesh(nr, nz, re.ctypes.data, ze.ctypes.data, 1 if spherical else 0)
        total = C.c_double(0.0)
        cnt = _Counts()
        rc = self.lib.vrc_next_event_rz(C.byref(self._p), C.byref(g), n, r.ctypes.data, d.ctypes.data,
                                        C.cast(C.byref(total), C.c_void_p), C.cast(C.byref(dg), C.c_void_p),
                                        C.cast(C.byref(cnt), C.c_void_p))
        if rc < 0:
            raise RuntimeError(f"oracle error {rc}")
        return NextEventResult(float(total.value), int(cnt.rays_accepted), int(cnt.rays_rejected), int(cnt.segments),
                               nseg, hsh, tau, score)

    def next_event_rz(self, rays, det, re, ze) -> NextEventResult:
        """Next-event estimator of `rays` for ONE detector point on the R-Z mesh (re, ze): steps NZ1..NZ6 of vrc_oracle.c."""
        return self._next_event_rz(rays, det, re, ze, False)

    def next_event_sphere(self, rays, det, re) -> NextEventResult:
        """The same on 1-D spherical shells about the origin."""
        return self._next_event_rz(rays, det, re, np.array([0.0, 1.0]), True)


# ---------------------------------------------------------------------------------------------------
# Per-batch moments: Eq. (5) FOM = 1/(sigma^2 T) with "sigma the
# standard deviation of the tally mean".  Plain numpy, fp64, one statement per definition.
# ---------------------------------------------------------------------------------------------------
def batch_moments(batch_tallies):
    """batch_tallies [B, ncell] (the tally of each batch on its own) -> (sum_b x_b, sum_b x_b^2) per cell."""
    x = np.asarray(batch_tallies, dtype=np.float64)
    s1 = np.zeros(x.shape[1])
    s2 = np.zeros(x.shape[1])
    for b in range(x.shape[0]):           # batch order, one add per batch (the order the device folds in)
        s1 = s1 + x[b]
        s2 = s2 + x[b] * x[b]
    return s1, s2


def mean_and_sigma(s1, s2, B: int):
    """Batch mean and the standard deviation OF THE MEAN per cell:
    mean = s1/B;  sigma^2 = (s2/B - mean^2) / (B - 1)  (unbiased sample variance / B), clamped at 0."""
    mean = s1 / B
    var = (s2 / B - mean * mean) / (B - 1) if B > 1 else np.full_like(mean, np.inf)
    return mean, np.sqrt(np.maximum(var, 0.0))


def figure_of_merit(sigma, T: float):
    """PAPER.md:93 Eq. (5): FOM = 1 / (sigma^2 T)."""
    return 1.0 / (sigma * sigma * T)


def fom_ratio(sigma_a, T_a: float, sigma_b, T_b: float):
    """PAPER.md:97 Eq. (6): eta = FOM_a / FOM_b = (sigma_b^2 / sigma_a^2) * (T_b / T_a)."""
    return (sigma_b * sigma_b) / (sigma_a * sigma_a) * (T_b / T_a)


def relative_difference(phi_ref, phi):
    """PAPER.md:118 Eq. (7): Delta_phi(i) = |phi_ref(i) - phi(i)| / phi_ref(i), the paper's measure of single-precision ray casting
    on the GPU against double precision on the CPU (phi_ref); cells with phi_ref = 0 give 0 where phi = 0 too, else +inf."""
    a, b = np.asarray(phi_ref, dtype=np.float64), np.asarray(phi, dtype=np.float64)
    d = np.abs(a - b)
    out = np.zeros_like(d)
    nz = a != 0.0
    out[nz] = d[nz] / np.abs(a[nz])
    out[~nz & (d > 0.0)] = np.inf
    return out


def fractional_difference(phi_ref, phi, sigma):
    """PAPER.md:122 Eq. (8): eps_phi(i) = |phi_ref(i) - phi(i)| / sigma(i), "the ratio of the absolute difference to the standard
    deviation of the fluence": whether a difference is statistically significant.  sigma = 0 gives 0 for equal values, else +inf."""
    a, b, s = (np.asarray(v, dtype=np.float64) for v in (phi_ref, phi, sigma))
    d = np.abs(a - b)
    out = np.zeros_like(d)
    nz = s > 0.0
    out[nz] = d[nz] / s[nz]
    out[~nz & (d > 0.0)] = np.inf
    return out
