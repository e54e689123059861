"""Thin ctypes binding of libmonteray.so (include/monteray.h): argument marshalling only.

Every step of the hot path runs inside the CUDA library; this module converts numpy / torch
arguments to pointers and sizes and turns status codes into exceptions.  PyTorch supplies
device memory (through the allocator callbacks) and the CUDA stream.  There is no CPU
fallback: if the shared library is missing or no CUDA device is usable, calls raise.
"""
from __future__ import annotations

import ctypes as C
import os
from dataclasses import dataclass
from typing import Optional

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libmonteray.so")

MR_OK, MR_ERR_INVALID_ARG, MR_ERR_STATE, MR_ERR_CUDA, MR_ERR_OOM, MR_ERR_UNSUPPORTED = range(6)
MR_PRECISION_MIXED, MR_PRECISION_DOUBLE = 0, 1
MR_WHERE_HOST, MR_WHERE_DEVICE = 0, 1
MR_STATIC_MAX_RAYS = 1 << 18
MR_OPT_BLOCK_THREADS, MR_OPT_SORT_RAYS, MR_OPT_STAGE_RAYS, MR_OPT_COPY_THREADS, MR_OPT_PAIR_RECORDS = 1, 2, 3, 4, 5
MR_OPT_ORDER_MODE = 6
MR_OPT_FUSED_TALLY = 7
MR_OPT_TILED_INDEX = 8
MR_OPT_AGGREGATE_FIRST = 9
MR_OPT_COARSE_RECORDS = 10
MR_OPT_DEFERRED_TALLY = 11
MR_OPT_DEFER_POOL_ENTRIES = 12
MR_OPT_DEFER_REGION_SHIFT = 13
MR_OPT_COOP_FLUSH = 14
MR_OPT_RZ_BLOCK_THREADS = 15
MR_OPT_TILED_TALLY = 16
MR_OPT_WHOLE_BATCH = 18
MR_OPT_RING_MERGE = 19
MR_INFO_RECORD_PATH, MR_INFO_DISTINCT_RECORDS, MR_INFO_COARSE_SHIFT = 100, 101, 102
MR_INFO_DEFERRED, MR_INFO_DEFER_DIRECT_PAIRS = 103, 104
MR_PATH_NAMES = {0: "none", 1: "k1", 2: "k2", 3: "k3", 4: "k4", 5: "k2_pairs", 6: "k3_pairs", 7: "k4_fused", 8: "dense8",
                 9: "generic", 10: "tiled4", 11: "tiled8", 12: "tiled16", 13: "coarse_blocks", 14: "double_k3",
                 15: "double_generic", 16: "rz"}
_STATUS = {1: "MR_ERR_INVALID_ARG", 2: "MR_ERR_STATE", 3: "MR_ERR_CUDA", 4: "MR_ERR_OOM", 5: "MR_ERR_UNSUPPORTED"}

EXPORTS = [
    "mr_create", "mr_create_ex", "mr_destroy", "mr_set_stream", "mr_last_error", "mr_load_mesh",
    "mr_load_materials", "mr_load_xs", "mr_cast_rays", "mr_cast_rays_static", "mr_read_tally", "mr_read_tally_async", "mr_clear_tally", "mr_sync",
    "mr_get_stats", "mr_tally_device_ptr", "mr_trace_rays", "mr_set_option", "mr_get_option",
    "mr_end_batch", "mr_read_moments", "mr_read_mean_sigma", "mr_load_nuclide_xs", "mr_define_material", "mr_load_mesh_rz", "mr_load_mesh_sphere",
    "mr_ring_open", "mr_ring_push", "mr_ring_flush", "mr_ring_close", "mr_ring_get_stats", "mr_ring_bench_producers",
    "mr_load_detectors", "mr_cast_next_event", "mr_read_detectors", "mr_clear_detectors", "mr_trace_next_event",
    "mr_microbench_red",
]


class MonteRayError(RuntimeError):
    def __init__(self, status: int, message: str):
        super().__init__(f"{_STATUS.get(status, status)}: {message}")
        self.status = status


class mr_stats(C.Structure):
    _fields_ = [("rays_accepted", C.c_int64), ("rays_rejected", C.c_int64), ("segments", C.c_int64),
                ("kernel_launches", C.c_int64), ("last_cast_ms", C.c_double), ("last_kernel_ms", C.c_double),
                ("ne_pairs_accepted", C.c_int64), ("ne_pairs_rejected", C.c_int64), ("ne_segments", C.c_int64)]


class mr_ring_stats(C.Structure):
    _fields_ = [("rays_pushed", C.c_int64), ("slots_shipped", C.c_int64), ("producer_wait_ms", C.c_double),
                ("casts", C.c_int64), ("reserved", C.c_double * 2)]


_ALLOC_FN = C.CFUNCTYPE(C.c_void_p, C.c_void_p, C.c_size_t, C.c_int)
_FREE_FN = C.CFUNCTYPE(None, C.c_void_p, C.c_void_p, C.c_int)


class mr_allocator(C.Structure):
    _fields_ = [("alloc", _ALLOC_FN), ("free", _FREE_FN), ("user", C.c_void_p)]


_lib = None


def load_library() -> C.CDLL:
    """Loads libmonteray.so; raises if it has not been built (python -m paper_1706_07476_b200.build)."""
    global _lib
    if _lib is not None:
        return _lib
    if not os.path.exists(LIB_PATH):
        raise ImportError(f"{LIB_PATH} not found: build it with `python -m paper_1706_07476_b200.build` "
                          "(there is no CPU fallback)")
    lib = C.CDLL(LIB_PATH)
    vp, i32, i64 = C.c_void_p, C.c_int, C.c_int64
    sigs = {
        "mr_create": [C.POINTER(vp), i32, i32],
        "mr_create_ex": [C.POINTER(vp), i32, i32, C.POINTER(mr_allocator)],
        "mr_destroy": [vp],
        "mr_set_stream": [vp, vp],
        "mr_load_mesh": [vp, i32, i32, i32, vp, vp, vp],
        "mr_load_mesh_rz": [vp, i32, i32, vp, vp],
        "mr_load_mesh_sphere": [vp, i32, vp],
        "mr_load_materials": [vp, i32, vp, i32, vp, vp],
        "mr_load_xs": [vp, i32, i64, vp, vp],
        "mr_cast_rays": [vp, i64, vp, i32],
        "mr_cast_rays_static": [vp, i64, vp],
        "mr_read_tally": [vp, vp],
        "mr_read_tally_async": [vp, vp],
        "mr_clear_tally": [vp],
        "mr_sync": [vp],
        "mr_get_stats": [vp, C.POINTER(mr_stats)],
        "mr_tally_device_ptr": [vp, C.POINTER(vp)],
        "mr_trace_rays": [vp, i64, vp, i32, vp, vp, vp, vp, i64],
        "mr_set_option": [vp, i32, i64],
        "mr_get_option": [vp, i32, C.POINTER(i64)],
        "mr_ring_open": [vp, i32, i64],
        "mr_ring_push": [vp, i64, vp],
        "mr_ring_flush": [vp],
        "mr_ring_close": [vp],
        "mr_ring_get_stats": [vp, C.POINTER(mr_ring_stats)],
        "mr_ring_bench_producers": [vp, i64, vp, i32, i64, i32, C.POINTER(C.c_double)],
        "mr_load_nuclide_xs": [vp, i32, i64, vp, vp],
        "mr_define_material": [vp, i32, i32, vp, vp],
        "mr_end_batch": [vp],
        "mr_read_moments": [vp, vp, vp, C.POINTER(i64)],
        "mr_read_mean_sigma": [vp, vp, vp, C.POINTER(i64)],
        "mr_load_detectors": [vp, i32, vp],
        "mr_cast_next_event": [vp, i64, vp, i32],
        "mr_read_detectors": [vp, vp],
        "mr_clear_detectors": [vp],
        "mr_trace_next_event": [vp, i64, vp, i32, i32, vp, vp, vp, vp],
        "mr_microbench_red": [i32, i64, i32, i32, i64, i32, C.POINTER(C.c_double), C.POINTER(C.c_double)],
    }
    for name, argtypes in sigs.items():
        fn = getattr(lib, name)
        fn.argtypes = argtypes
        fn.restype = C.c_int
    lib.mr_last_error.argtypes = [vp]
    lib.mr_last_error.restype = C.c_char_p
    _lib = lib
    return lib


def microbench_red(device: int, ncell: int, group: int = 1, gather_bytes: int = 0, lane_ops: int = 1 << 28, reps: int = 5):
    """mr_microbench_red -> dict(lane_ops, best_ms, mean_ms, lane_ops_per_sec): the L2 fp64-atomic ceiling."""
    lib = load_library()
    best, mean = C.c_double(), C.c_double()
    rc = lib.mr_microbench_red(device, ncell, group, gather_bytes, lane_ops, reps, C.byref(best), C.byref(mean))
    if rc != MR_OK:
        raise MonteRayError(rc, "mr_microbench_red failed")
    ops = max(128, (lane_ops + 63) // 64 // 128 * 128) * 64
    return {"ncell": int(ncell), "group": group, "gather_bytes": gather_bytes, "lane_ops": ops, "best_ms": best.value,
            "mean_ms": mean.value, "lane_ops_per_sec": ops / (best.value * 1e-3)}


class _TorchAllocator:
    """mr_allocator backed by torch's CUDA caching allocator (uint8 tensors kept alive by pointer)."""

    def __init__(self):
        import torch

        self._torch = torch
        self._live = {}
        self._alloc_cb = _ALLOC_FN(self._alloc)
        self._free_cb = _FREE_FN(self._free)
        self.struct = mr_allocator(self._alloc_cb, self._free_cb, None)

    def _alloc(self, user, nbytes, device):
        try:
            t = self._torch.empty(max(int(nbytes), 16), dtype=self._torch.uint8, device=f"cuda:{device}")
        except Exception:  # out of memory -> NULL -> MR_ERR_OOM
            return None
        self._live[t.data_ptr()] = t
        return t.data_ptr()

    def _free(self, user, ptr, device):
        self._live.pop(ptr, None)


@dataclass
class Stats:
    rays_accepted: int
    rays_rejected: int
    segments: int
    kernel_launches: int
    last_cast_ms: float
    last_kernel_ms: float
    ne_pairs_accepted: int = 0
    ne_pairs_rejected: int = 0
    ne_segments: int = 0


def _f64(a) -> np.ndarray:
    return np.ascontiguousarray(a, dtype=np.float64)


class MonteRay:
    """One library context.  Method names mirror the C entry points (mr_<name>)."""

    def __init__(self, device: int = 0, precision: int = MR_PRECISION_MIXED, use_torch_allocator: bool = True,
                 use_torch_stream: bool = True):
        self.lib = load_library()
        self.precision = precision
        self.device = device
        self._h = C.c_void_p()
        self._allocator = None
        if use_torch_allocator:
            import torch

            if not torch.cuda.is_available():
                raise MonteRayError(MR_ERR_CUDA, "no CUDA device visible to torch (there is no CPU fallback)")
            torch.cuda.init()
            self._allocator = _TorchAllocator()
            rc = self.lib.mr_create_ex(C.byref(self._h), device, precision, C.byref(self._allocator.struct))
        else:
            rc = self.lib.mr_create(C.byref(self._h), device, precision)
        if rc != MR_OK:
            raise MonteRayError(rc, (self.lib.mr_last_error(None) or b"").decode())
        self.ncell = 0
        if use_torch_stream:
            self.use_current_torch_stream()

    # ---- plumbing
    def _check(self, rc: int):
        if rc != MR_OK:
            raise MonteRayError(rc, (self.lib.mr_last_error(self._h) or b"").decode())

    def close(self):
        if self._h:
            self.lib.mr_destroy(self._h)
            self._h = C.c_void_p()

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def __enter__(self):
        return self

    def __exit__(self, *exc):
        self.close()

    def use_current_torch_stream(self):
        import torch

        self.set_stream(torch.cuda.current_stream(self.device).cuda_stream)

    def set_stream(self, cuda_stream: int):
        self._check(self.lib.mr_set_stream(self._h, C.c_void_p(cuda_stream)))

    @property
    def ray_dtype(self):
        return np.float64 if self.precision == MR_PRECISION_DOUBLE else np.float32

    # ---- set-up
    def load_mesh(self, xe, ye, ze):
        xe, ye, ze = _f64(xe), _f64(ye), _f64(ze)
        self._check(self.lib.mr_load_mesh(self._h, len(xe) - 1, len(ye) - 1, len(ze) - 1,
                                          xe.ctypes.data, ye.ctypes.data, ze.ctypes.data))
        self.ncell = (len(xe) - 1) * (len(ye) - 1) * (len(ze) - 1)

    def load_mesh_rz(self, re, ze):
        re, ze = _f64(re), _f64(ze)
        self._check(self.lib.mr_load_mesh_rz(self._h, len(re) - 1, len(ze) - 1, re.ctypes.data, ze.ctypes.data))
        self.ncell = (len(re) - 1) * (len(ze) - 1)

    def load_mesh_sphere(self, re):
        re = _f64(re)
        self._check(self.lib.mr_load_mesh_sphere(self._h, len(re) - 1, re.ctypes.data))
        self.ncell = len(re) - 1

    def load_materials(self, density, cell_mat, cell_frac):
        density = _f64(density)
        cell_mat = np.ascontiguousarray(cell_mat, dtype=np.int32)
        cell_frac = _f64(cell_frac)
        if cell_mat.size != cell_frac.size or self.ncell == 0 or cell_mat.size % self.ncell:
            raise MonteRayError(MR_ERR_INVALID_ARG, "cell_mat / cell_frac must both hold ncell*K entries")
        K = cell_mat.size // self.ncell
        self._check(self.lib.mr_load_materials(self._h, len(density), density.ctypes.data, K,
                                               cell_mat.ctypes.data, cell_frac.ctypes.data))

    def load_xs(self, material: int, energy, sigma_t):
        energy, sigma_t = _f64(energy), _f64(sigma_t)
        if len(energy) != len(sigma_t):
            raise MonteRayError(MR_ERR_INVALID_ARG, "energy and sigma_t differ in length")
        self._check(self.lib.mr_load_xs(self._h, material, len(energy), energy.ctypes.data, sigma_t.ctypes.data))

    def load_nuclide_xs(self, nuclide: int, energy, sigma):
        energy, sigma = _f64(energy), _f64(sigma)
        if len(energy) != len(sigma):
            raise MonteRayError(MR_ERR_INVALID_ARG, "energy and sigma differ in length")
        self._check(self.lib.mr_load_nuclide_xs(self._h, nuclide, len(energy), energy.ctypes.data, sigma.ctypes.data))

    def define_material(self, material: int, nuclides, weights):
        nuclides = np.ascontiguousarray(nuclides, dtype=np.int32)
        weights = _f64(weights)
        if len(nuclides) != len(weights):
            raise MonteRayError(MR_ERR_INVALID_ARG, "nuclides and weights differ in length")
        self._check(self.lib.mr_define_material(self._h, material, len(nuclides), nuclides.ctypes.data, weights.ctypes.data))

    def load_problem(self, prob):
        """Convenience: mesh + materials + all tables (and nuclide mixtures) of a workloads.Problem-like object."""
        if getattr(prob, "sphere", False):
            self.load_mesh_sphere(prob.re)
        elif getattr(prob, "re", None) is not None:
            self.load_mesh_rz(prob.re, prob.ze)
        else:
            self.load_mesh(prob.xe, prob.ye, prob.ze)
        self.load_materials(prob.density, prob.cell_mat, prob.cell_frac)
        mixtures = getattr(prob, "mixtures", None) or [None] * len(prob.xs)
        for q, (e, s) in enumerate(getattr(prob, "nuclide_xs", None) or []):
            self.load_nuclide_xs(q, e, s)
        for m, t in enumerate(prob.xs):
            if mixtures[m] is not None:
                self.define_material(m, *mixtures[m])
            else:
                self.load_xs(m, *t)

    # ---- hot path
    def _ray_arg(self, rays):
        """(pointer, n, where, keepalive) for a numpy array (host) or a torch CUDA tensor (device)."""
        if isinstance(rays, np.ndarray):
            a = np.ascontiguousarray(rays, dtype=self.ray_dtype).reshape(-1, 8)
            return a.ctypes.data, a.shape[0], MR_WHERE_HOST, a
        import torch

        if isinstance(rays, torch.Tensor):
            want = torch.float64 if self.precision == MR_PRECISION_DOUBLE else torch.float32
            if rays.dtype != want or not rays.is_contiguous() or rays.numel() % 8:
                raise MonteRayError(MR_ERR_INVALID_ARG, f"ray tensor must be contiguous {want} with 8 fields per ray")
            n = rays.numel() // 8
            if rays.is_cuda:
                return rays.data_ptr(), n, MR_WHERE_DEVICE, rays
            return rays.data_ptr(), n, MR_WHERE_HOST, rays  # CPU tensor (pinned or pageable)
        raise MonteRayError(MR_ERR_INVALID_ARG, "rays must be a numpy array or a torch tensor")

    def cast_rays(self, rays):
        ptr, n, where, keep = self._ray_arg(rays)
        self._check(self.lib.mr_cast_rays(self._h, n, C.c_void_p(ptr), where))
        return n

    def cast_rays_static(self, rays):
        """mr_cast_rays_static: casts a torch CUDA tensor of at most MR_STATIC_MAX_RAYS rays without allocating device
        memory (the ordering scratch is a fixed array in the library).  For hosts that own all device memory
        themselves or cannot stall on cudaMalloc inside their loop; see include/monteray.h for the rules."""
        ptr, n, where, keep = self._ray_arg(rays)
        if where != MR_WHERE_DEVICE:
            raise MonteRayError(MR_ERR_INVALID_ARG, "cast_rays_static takes device-resident rays (a torch CUDA tensor)")
        self._check(self.lib.mr_cast_rays_static(self._h, n, C.c_void_p(ptr)))
        return n

    def read_tally(self, out: Optional[np.ndarray] = None) -> np.ndarray:
        if out is None:
            out = np.empty(self.ncell, dtype=np.float64)
        assert out.dtype == np.float64 and out.size == self.ncell and out.flags.c_contiguous
        self._check(self.lib.mr_read_tally(self._h, out.ctypes.data))
        return out

    def read_tally_into(self, host_ptr: int):
        """mr_read_tally into caller-owned host memory (e.g. a pinned torch tensor's data_ptr())."""
        self._check(self.lib.mr_read_tally(self._h, C.c_void_p(host_ptr)))

    def read_tally_async_into(self, host_ptr: int):
        """mr_read_tally_async into caller-owned (page-locked) host memory; valid after sync()."""
        self._check(self.lib.mr_read_tally_async(self._h, C.c_void_p(host_ptr)))

    def clear_tally(self):
        self._check(self.lib.mr_clear_tally(self._h))

    def sync(self):
        self._check(self.lib.mr_sync(self._h))

    def get_stats(self) -> Stats:
        s = mr_stats()
        self._check(self.lib.mr_get_stats(self._h, C.byref(s)))
        return Stats(s.rays_accepted, s.rays_rejected, s.segments, s.kernel_launches, s.last_cast_ms, s.last_kernel_ms,
                     s.ne_pairs_accepted, s.ne_pairs_rejected, s.ne_segments)

    def tally_device_ptr(self) -> int:
        p = C.c_void_p()
        self._check(self.lib.mr_tally_device_ptr(self._h, C.byref(p)))
        return int(p.value)

    def tally_tensor(self):
        """The resident tally as a torch tensor view (no copy), e.g. for torch.distributed.all_reduce."""
        import torch

        class _Wrap:
            pass

        w = _Wrap()
        w.__cuda_array_interface__ = {"shape": (self.ncell,), "typestr": "<f8", "data": (self.tally_device_ptr(), False),
                                      "version": 3, "strides": None}
        return torch.as_tensor(w, device=f"cuda:{self.device}")

    def trace_rays(self, rays, cap: int = 0):
        """mr_trace_rays -> (nseg uint32[n], hash uint64[n], cells int32[n,cap] | None, lens float64[n,cap] | None)."""
        ptr, n, where, keep = self._ray_arg(rays)
        nseg = np.zeros(n, dtype=np.uint32)
        hsh = np.zeros(n, dtype=np.uint64)
        cells = np.full((n, cap), -1, dtype=np.int32) if cap > 0 else None
        lens = np.zeros((n, cap), dtype=np.float64) if cap > 0 else None
        self._check(self.lib.mr_trace_rays(self._h, n, C.c_void_p(ptr), where, nseg.ctypes.data, hsh.ctypes.data,
                                           cells.ctypes.data if cap > 0 else None,
                                           lens.ctypes.data if cap > 0 else None, cap))
        return nseg, hsh, cells, lens

    # ---- producer ring (NEXT-1)
    def ring_open(self, slots: int, rays_per_slot: int):
        self._check(self.lib.mr_ring_open(self._h, slots, rays_per_slot))

    def ring_push(self, rays: np.ndarray):
        """mr_ring_push of a host array; thread-safe (ctypes releases the GIL for the duration of the call)."""
        a = rays if (isinstance(rays, np.ndarray) and rays.dtype == self.ray_dtype and rays.flags.c_contiguous) \
            else np.ascontiguousarray(rays, dtype=self.ray_dtype)
        rc = self.lib.mr_ring_push(self._h, a.size // 8, C.c_void_p(a.ctypes.data))
        if rc != MR_OK:
            raise MonteRayError(rc, "mr_ring_push failed")

    def ring_flush(self):
        self._check(self.lib.mr_ring_flush(self._h))

    def ring_close(self):
        self._check(self.lib.mr_ring_close(self._h))

    def ring_stats(self):
        s = mr_ring_stats()
        self._check(self.lib.mr_ring_get_stats(self._h, C.byref(s)))
        return {"rays_pushed": int(s.rays_pushed), "slots_shipped": int(s.slots_shipped),
                "producer_wait_ms": float(s.producer_wait_ms), "casts": int(s.casts)}

    def ring_bench_producers(self, rays, producers: int, rays_per_push: int, dry_run: bool = False) -> float:
        """mr_ring_bench_producers: library-side producer threads push the host batch through the ring; wall ms."""
        rays = np.ascontiguousarray(rays, dtype=self.ray_dtype)
        ms = C.c_double(0.0)
        self._check(self.lib.mr_ring_bench_producers(self._h, rays.size // 8, rays.ctypes.data_as(C.c_void_p), int(producers),
                                                     int(rays_per_push), 1 if dry_run else 0, C.byref(ms)))
        return float(ms.value)

    # ---- per-batch moments (NEXT-2)
    def end_batch(self):
        self._check(self.lib.mr_end_batch(self._h))

    def read_moments(self):
        """mr_read_moments -> (sum float64[ncell], sumsq float64[ncell], nbatch)."""
        s1 = np.empty(self.ncell, dtype=np.float64)
        s2 = np.empty(self.ncell, dtype=np.float64)
        nb = C.c_int64()
        self._check(self.lib.mr_read_moments(self._h, s1.ctypes.data, s2.ctypes.data, C.byref(nb)))
        return s1, s2, int(nb.value)

    def read_mean_sigma(self):
        """mr_read_mean_sigma -> (mean float64[ncell], sigma float64[ncell], nbatch)."""
        mean = np.empty(self.ncell, dtype=np.float64)
        sigma = np.empty(self.ncell, dtype=np.float64)
        nb = C.c_int64()
        self._check(self.lib.mr_read_mean_sigma(self._h, mean.ctypes.data, sigma.ctypes.data, C.byref(nb)))
        return mean, sigma, int(nb.value)

    # ---- next-event estimator (NEXT-3)
    def load_detectors(self, xyz):
        xyz = _f64(xyz).reshape(-1, 3)
        self._check(self.lib.mr_load_detectors(self._h, xyz.shape[0], xyz.ctypes.data))
        self.ndet = xyz.shape[0]

    def cast_next_event(self, rays):
        ptr, n, where, keep = self._ray_arg(rays)
        self._check(self.lib.mr_cast_next_event(self._h, n, C.c_void_p(ptr), where))
        return n

    def read_detectors(self) -> np.ndarray:
        out = np.empty(self.ndet, dtype=np.float64)
        self._check(self.lib.mr_read_detectors(self._h, out.ctypes.data))
        return out

    def clear_detectors(self):
        self._check(self.lib.mr_clear_detectors(self._h))

    def trace_next_event(self, rays, det: int):
        """mr_trace_next_event -> (nseg uint32[n], hash uint64[n], tau float64[n], score float64[n])."""
        ptr, n, where, keep = self._ray_arg(rays)
        nseg = np.zeros(n, dtype=np.uint32)
        hsh = np.zeros(n, dtype=np.uint64)
        tau = np.zeros(n, dtype=np.float64)
        score = np.zeros(n, dtype=np.float64)
        self._check(self.lib.mr_trace_next_event(self._h, n, C.c_void_p(ptr), where, det, nseg.ctypes.data,
                                                 hsh.ctypes.data, tau.ctypes.data, score.ctypes.data))
        return nseg, hsh, tau, score

    def record_path(self) -> str:
        """Name of the cell-record path mr_cast_rays takes for the resident problem (MR_INFO_RECORD_PATH)."""
        return MR_PATH_NAMES[self.get_option(MR_INFO_RECORD_PATH)]

    def set_option(self, option: int, value: int):
        self._check(self.lib.mr_set_option(self._h, option, value))

    def get_option(self, option: int) -> int:
        v = C.c_int64()
        self._check(self.lib.mr_get_option(self._h, option, C.byref(v)))
        return int(v.value)
