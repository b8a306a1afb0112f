"""ctypes binding of libamrgodunov.so -- argument marshalling only (include/amr_godunov.h has the
contract).  Every step of the hot path runs inside the library's CUDA kernels; nothing here computes.

torch is imported lazily and used for exactly two things: the device arena (a uint8 tensor the
library borrows) and the current CUDA stream handle.
"""
from __future__ import annotations

import ctypes as C
import os
from typing import Optional, Sequence

import numpy as np

AMR_F32, AMR_F64 = 0, 1
AMR_BC_PERIODIC, AMR_BC_OUTFLOW = 0, 1
AMR_LIM_NONE, AMR_LIM_MINMOD, AMR_LIM_MC = 0, 1, 2
AMR_RS_HLL, AMR_RS_HLLC, AMR_RS_HLLD = 0, 1, 2
CNT_NAMES = ("positivity_fallback_cells", "hll_fallback_faces", "degenerate_D", "nonpositive_rho_after")

# every symbol include/amr_godunov.h declares
EXPORTS = (
    "amr_patch_batch_bytes", "amr_patch_batch_create", "amr_patch_batch_destroy", "amr_patch_batch_upload",
    "amr_patch_batch_download", "amr_patch_batch_state", "amr_fill_ghosts", "amr_cfl_dt", "amr_hydro_step",
    "amr_mhd_step", "amr_conserved_totals", "amr_step_counters", "amr_link_bytes", "amr_link_levels",
    "amr_link_destroy", "amr_prolong_ghosts", "amr_flux_clear", "amr_restrict", "amr_reflux", "amr_last_error",
    "amr_version", "amr_builder_bytes", "amr_builder_create", "amr_builder_destroy", "amr_builder_build",
    "amr_builder_results", "amr_builder_gather", "amr_hierarchy_cfl_dt", "amr_hierarchy_step",
    "amr_flag_blocks", "amr_regrid_bytes", "amr_regrid_fill", "amr_measure_fma_peak", "amr_hydro_sweep_ppm",
    "amr_hydro_step_ppm", "amr_patch_batch_export", "amr_patch_batch_import", "amr_conserved_totals_noalloc",
)


class AmrError(RuntimeError):
    def __init__(self, code: int, msg: str):
        super().__init__("amr_godunov error %d: %s" % (code, msg))
        self.code = code


class _Desc(C.Structure):
    _fields_ = [("npatch", C.c_int32), ("n", C.c_int32), ("nghost", C.c_int32), ("nfields", C.c_int32),
                ("dtype", C.c_int32), ("level", C.c_int32), ("dx", C.c_double), ("origin", C.c_void_p),
                ("domain_cells", C.c_int32 * 3), ("bc", C.c_int32 * 6), ("self_periodic", C.c_int32),
                ("nactive", C.c_int32)]


_lib = None


def library_path() -> str:
    return os.path.join(os.path.dirname(os.path.abspath(__file__)), "libamrgodunov.so")


def lib():
    """Load the C-ABI library.  Fails loudly if it has not been built (no fallback of any kind)."""
    global _lib
    if _lib is None:
        path = library_path()
        if not os.path.exists(path):
            raise ImportError("%s is missing: run `python -m paper_1412_0934_b200.build` (needs nvcc)" % path)
        L = C.CDLL(path)
        L.amr_last_error.restype = C.c_char_p
        L.amr_version.restype = C.c_char_p
        L.amr_patch_batch_bytes.restype = C.c_size_t
        L.amr_patch_batch_bytes.argtypes = [C.POINTER(_Desc)]
        L.amr_patch_batch_create.argtypes = [C.POINTER(_Desc), C.c_void_p, C.c_size_t, C.c_void_p, C.POINTER(C.c_void_p)]
        L.amr_patch_batch_destroy.argtypes = [C.c_void_p]
        L.amr_patch_batch_upload.argtypes = [C.c_void_p, C.c_void_p, C.c_int]
        L.amr_patch_batch_download.argtypes = [C.c_void_p, C.c_void_p, C.c_int]
        L.amr_patch_batch_state.restype = C.c_void_p
        L.amr_patch_batch_state.argtypes = [C.c_void_p, C.c_int]
        L.amr_fill_ghosts.argtypes = [C.c_void_p]
        L.amr_cfl_dt.argtypes = [C.c_void_p, C.c_double, C.c_double, C.c_int, C.POINTER(C.c_double), C.POINTER(C.c_double)]
        L.amr_hydro_step.argtypes = [C.c_void_p, C.c_double, C.c_double, C.c_int, C.c_int]
        L.amr_mhd_step.argtypes = [C.c_void_p, C.c_double, C.c_double, C.c_int, C.c_int, C.c_double, C.c_double]
        L.amr_conserved_totals.argtypes = [C.c_void_p, C.c_void_p]
        L.amr_conserved_totals_noalloc.argtypes = [C.c_void_p, C.c_int, C.c_int, C.c_int64, C.c_int64, C.c_void_p, C.c_void_p]
        L.amr_step_counters.argtypes = [C.c_void_p, C.c_void_p, C.c_int]
        L.amr_link_bytes.restype = C.c_size_t
        L.amr_link_bytes.argtypes = [C.c_void_p, C.c_void_p, C.c_int]
        L.amr_link_levels.argtypes = [C.c_void_p, C.c_void_p, C.c_int, C.c_void_p, C.c_size_t, C.POINTER(C.c_void_p)]
        L.amr_link_destroy.argtypes = [C.c_void_p]
        L.amr_prolong_ghosts.argtypes = [C.c_void_p, C.c_double]
        L.amr_flux_clear.argtypes = [C.c_void_p]
        L.amr_restrict.argtypes = [C.c_void_p]
        L.amr_reflux.argtypes = [C.c_void_p, C.c_double]
        L.amr_builder_bytes.restype = C.c_size_t
        L.amr_builder_bytes.argtypes = [C.c_int64]
        L.amr_builder_create.argtypes = [C.c_int64, C.c_void_p, C.c_size_t, C.c_void_p, C.POINTER(C.c_void_p)]
        L.amr_builder_destroy.argtypes = [C.c_void_p]
        L.amr_builder_build.argtypes = [C.c_void_p, C.c_void_p, C.c_int64, C.c_int32, C.c_int32, C.POINTER(C.c_int64)]
        L.amr_builder_results.argtypes = [C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p]
        L.amr_flag_blocks.argtypes = [C.c_void_p, C.c_int, C.c_double, C.c_void_p]
        L.amr_regrid_bytes.argtypes = [C.c_void_p, C.c_void_p, C.c_void_p]
        L.amr_regrid_bytes.restype = C.c_size_t
        L.amr_regrid_fill.argtypes = [C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p, C.c_size_t]
        L.amr_hierarchy_cfl_dt.argtypes = [C.POINTER(C.c_void_p), C.c_int, C.c_double, C.c_double, C.c_int,
                                           C.POINTER(C.c_double), C.POINTER(C.c_double)]
        L.amr_hierarchy_step.argtypes = [C.POINTER(C.c_void_p), C.POINTER(C.c_void_p), C.c_int, C.c_int, C.c_double,
                                         C.c_double, C.c_int, C.c_int, C.c_double, C.c_double, C.c_int]
        L.amr_builder_gather.argtypes = [C.c_void_p, C.c_void_p, C.c_int32, C.c_int32, C.c_int32, C.c_void_p, C.c_int64,
                                         C.c_void_p, C.POINTER(C.c_int64)]
        L.amr_hydro_sweep_ppm.argtypes = [C.c_void_p, C.c_double, C.c_double, C.c_int, C.c_int]
        L.amr_hydro_step_ppm.argtypes = [C.c_void_p, C.c_double, C.c_double, C.c_int, C.c_int]
        L.amr_patch_batch_export.argtypes = [C.c_void_p, C.c_void_p, C.c_int32, C.c_void_p]
        L.amr_patch_batch_import.argtypes = [C.c_void_p, C.c_void_p, C.c_int32, C.c_void_p]
        L.amr_measure_fma_peak.argtypes = [C.c_int32, C.c_void_p, C.c_void_p, C.c_double, C.POINTER(C.c_double)]
        _lib = L
    return _lib


def _check(rc: int):
    if rc != 0:
        raise AmrError(rc, lib().amr_last_error().decode())


def measure_fma_peak(dtype: int, ms_target: float = 2.0, device: str = "cuda:0") -> float:
    """amr_measure_fma_peak: plain FMA throughput of the device in TFLOP/s (the benchmark's measured ALU peak)."""
    import torch
    scratch = torch.zeros(64, dtype=torch.uint8, device=device)
    out = C.c_double()
    with torch.cuda.device(scratch.device):
        _check(lib().amr_measure_fma_peak(dtype, scratch.data_ptr(), int(torch.cuda.current_stream().cuda_stream),
                                          float(ms_target), C.byref(out)))
    return float(out.value)


def conserved_totals_noalloc(dev_U, nfields: int, ncells: int, field_stride: int, dev_totals, dtype: int = None,
                             stream: int = None):
    """amr_conserved_totals_noalloc: dev_U / dev_totals are torch device tensors (or raw device addresses, then pass
    dtype); only enqueues on `stream` (default: torch's current stream of the tensor's device)."""
    import torch
    if isinstance(dev_U, torch.Tensor):
        if dtype is None:
            dtype = AMR_F64 if dev_U.dtype == torch.float64 else AMR_F32
        ctx, pu = torch.cuda.device(dev_U.device), dev_U.data_ptr()
    else:
        ctx, pu = torch.cuda.device(torch.cuda.current_device()), int(dev_U)
    pt = dev_totals.data_ptr() if isinstance(dev_totals, torch.Tensor) else int(dev_totals)
    with ctx:
        st = int(torch.cuda.current_stream().cuda_stream) if stream is None else int(stream)
        _check(lib().amr_conserved_totals_noalloc(pu, int(dtype), int(nfields), int(ncells), int(field_stride), pt, st))


def _np_dtype(dtype: int):
    return np.float64 if dtype == AMR_F64 else np.float32


def _host_ptr(a) -> int:
    """Host pointer of a C-contiguous numpy array or (pinned) CPU torch tensor."""
    if isinstance(a, np.ndarray):
        assert a.flags["C_CONTIGUOUS"]
        return a.ctypes.data
    assert a.device.type == "cpu" and a.is_contiguous()
    return a.data_ptr()


class PatchBatch:
    """amr_patch_batch: all equal-size patches of one level, resident in one device arena."""

    def __init__(self, npatch: int, n: int, nfields: int, dtype: int, dx: float, origin=None,
                 domain_cells: Sequence[int] = (0, 0, 0), bc: Sequence[int] = (0,) * 6, self_periodic: bool = False,
                 nghost: int = 3, level: int = 0, device: str = "cuda:0", stream: Optional[int] = None,
                 nactive: int = 0):
        import torch  # device memory + stream only
        self._torch = torch
        L = lib()
        d = _Desc()
        d.npatch, d.n, d.nghost, d.nfields, d.dtype, d.level, d.dx = npatch, n, nghost, nfields, dtype, level, dx
        self._origin = None
        if origin is not None:
            self._origin = np.ascontiguousarray(np.asarray(origin, dtype=np.int32).reshape(-1, 3))
            if self._origin.shape[0] != npatch:
                raise ValueError("origin must be [npatch, 3]")
            d.origin = self._origin.ctypes.data
        d.domain_cells[:] = [int(v) for v in domain_cells]
        d.bc[:] = [int(v) for v in bc]
        d.self_periodic = int(bool(self_periodic))
        d.nactive = int(nactive)
        self.nactive = int(nactive) if nactive else int(npatch)
        self.npatch, self.n, self.nghost, self.nfields, self.dtype, self.dx, self.level = npatch, n, nghost, nfields, dtype, dx, level
        nbytes = L.amr_patch_batch_bytes(C.byref(d))
        if nbytes == 0:
            raise AmrError(-1, L.amr_last_error().decode())
        self.device = torch.device(device)
        with torch.cuda.device(self.device):
            self.arena = torch.empty(nbytes, dtype=torch.uint8, device=self.device)  # borrowed by the library
            self.stream = int(torch.cuda.current_stream().cuda_stream) if stream is None else int(stream)
            h = C.c_void_p()
            _check(L.amr_patch_batch_create(C.byref(d), self.arena.data_ptr(), nbytes, self.stream, C.byref(h)))
        self._h = h
        self.arena_bytes = int(nbytes)

    @classmethod
    def from_level(cls, level, dtype: int, **kw):
        """Build from a workloads.Level (plain data) and upload its interiors."""
        b = cls(level.npatch, level.n, level.nfields, dtype, level.dx, origin=level.origin,
                domain_cells=level.domain_cells, bc=level.bc, self_periodic=level.self_periodic, nghost=level.g,
                level=level.level, **kw)
        b.upload(np.ascontiguousarray(level.U.astype(_np_dtype(dtype))))
        return b

    @property
    def handle(self):
        return self._h

    @property
    def np_dtype(self):
        return _np_dtype(self.dtype)

    @property
    def ncells(self) -> int:
        return self.npatch * self.n ** 3

    def _shape(self, with_ghosts: bool):
        m = self.n + (2 * self.nghost if with_ghosts else 0)
        return (self.nfields, self.npatch, m, m, m)

    def upload(self, host, with_ghosts: bool = False):
        assert tuple(host.shape) == self._shape(with_ghosts), (tuple(host.shape), self._shape(with_ghosts))
        _check(lib().amr_patch_batch_upload(self._h, _host_ptr(host), int(with_ghosts)))

    def download(self, with_ghosts: bool = False, out=None):
        if out is None:
            out = np.empty(self._shape(with_ghosts), dtype=self.np_dtype)
        _check(lib().amr_patch_batch_download(self._h, _host_ptr(out), int(with_ghosts)))
        return out

    def export_patches(self, dev_pairs, count: int, dev_packed):
        """amr_patch_batch_export: dev_pairs int32 [count, 2] = (slot, patch), dev_packed [nfields, count, n^3]
        (device tensors)."""
        _check(lib().amr_patch_batch_export(self._h, dev_pairs.data_ptr(), int(count), dev_packed.data_ptr()))

    def import_patches(self, dev_pairs, count: int, dev_packed):
        _check(lib().amr_patch_batch_import(self._h, dev_pairs.data_ptr(), int(count), dev_packed.data_ptr()))

    def state_ptr(self, which: int = 0) -> int:
        return int(lib().amr_patch_batch_state(self._h, which))

    def fill_ghosts(self):
        _check(lib().amr_fill_ghosts(self._h))

    def cfl_dt(self, gamma: float, cfl: float):
        dt, sm = C.c_double(), C.c_double()
        _check(lib().amr_cfl_dt(self._h, gamma, cfl, int(self.nfields == 9), C.byref(dt), C.byref(sm)))
        return dt.value, sm.value

    def hydro_step(self, dt: float, gamma: float, limiter: int, riemann: int):
        _check(lib().amr_hydro_step(self._h, dt, gamma, limiter, riemann))

    def hydro_sweep_ppm(self, dt: float, gamma: float, riemann: int, direction: int):
        _check(lib().amr_hydro_sweep_ppm(self._h, dt, gamma, riemann, direction))

    def hydro_step_ppm(self, dt: float, gamma: float, riemann: int, order: int = 0):
        _check(lib().amr_hydro_step_ppm(self._h, dt, gamma, riemann, order))

    def mhd_step(self, dt: float, gamma: float, limiter: int, riemann: int, ch: float, alpha: float):
        _check(lib().amr_mhd_step(self._h, dt, gamma, limiter, riemann, ch, alpha))

    def conserved_totals(self) -> np.ndarray:
        out = np.zeros(self.nfields, dtype=np.float64)
        _check(lib().amr_conserved_totals(self._h, out.ctypes.data))
        return out

    def step_counters(self, reset: bool = False) -> dict:
        out = np.zeros(4, dtype=np.int64)
        _check(lib().amr_step_counters(self._h, out.ctypes.data, int(reset)))
        return dict(zip(CNT_NAMES, out.tolist()))

    def flag_blocks(self, field: int, threshold: float) -> np.ndarray:
        """amr_flag_blocks: bool [npatch, 2, 2, 2] (z, y, x halves of each patch)."""
        out = np.zeros(self.npatch * 8, dtype=np.uint8)
        _check(lib().amr_flag_blocks(self.handle, int(field), float(threshold), out.ctypes.data))
        return out.reshape(self.npatch, 2, 2, 2).astype(bool)

    def regrid_fill(self, old_fine, coarse):
        """amr_regrid_fill into this (new, not yet linked) fine batch."""
        import torch
        L = lib()
        oh = old_fine.handle if old_fine is not None else None
        nbytes = L.amr_regrid_bytes(self.handle, oh, coarse.handle)
        if nbytes == 0:
            raise AmrError(-1, L.amr_last_error().decode())
        ws = torch.empty(nbytes, dtype=torch.uint8, device=self.device)
        _check(L.amr_regrid_fill(self.handle, oh, coarse.handle, ws.data_ptr(), nbytes))

    def synchronize(self):
        self._torch.cuda.synchronize(self.device)

    def close(self):
        if self._h is not None and self._h.value:
            _check(lib().amr_patch_batch_destroy(self._h))
            self._h = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass


class LevelLink:
    """amr_level_link: coarse<->fine tables and flux registers (O8, O9)."""

    def __init__(self, coarse: PatchBatch, fine: PatchBatch, ratio: int = 2):
        import torch
        L = lib()
        nbytes = L.amr_link_bytes(coarse.handle, fine.handle, ratio)
        if nbytes == 0:
            raise AmrError(-1, L.amr_last_error().decode())
        self.coarse, self.fine = coarse, fine
        self.ws = torch.empty(nbytes, dtype=torch.uint8, device=coarse.device)
        h = C.c_void_p()
        _check(L.amr_link_levels(coarse.handle, fine.handle, ratio, self.ws.data_ptr(), nbytes, C.byref(h)))
        self._h = h
        self.ws_bytes = int(nbytes)

    def prolong_ghosts(self, theta: float):
        _check(lib().amr_prolong_ghosts(self._h, theta))

    def flux_clear(self):
        _check(lib().amr_flux_clear(self._h))

    def restrict(self):
        _check(lib().amr_restrict(self._h))

    def reflux(self, dt_coarse: float):
        _check(lib().amr_reflux(self._h, dt_coarse))

    def close(self):
        if self._h is not None and self._h.value:
            _check(lib().amr_link_destroy(self._h))
            self._h = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass


class Hierarchy:
    """L levels resident on the device + the links between consecutive levels;
    amr_hierarchy_cfl_dt / amr_hierarchy_step do the recursive subcycling."""

    def __init__(self, batches, mhd: bool):
        self.levels = list(batches)
        self.mhd = bool(mhd)
        self.links = [LevelLink(self.levels[l], self.levels[l + 1]) for l in range(len(self.levels) - 1)]
        self._tables()

    def _tables(self):
        n = len(self.levels)
        self._lv = (C.c_void_p * n)(*[b.handle for b in self.levels])
        self._lk = (C.c_void_p * max(n - 1, 1))(*[l._h for l in self.links])

    @classmethod
    def from_workload(cls, wl, dtype: int, **kw):
        return cls([PatchBatch.from_level(lv, dtype, **kw) for lv in wl.levels], wl.mhd)

    def replace_level(self, l: int, new_batch):
        """After a regrid: level l's batch is replaced by new_batch (already filled, amr_regrid_fill).  The links
        from level l-1 upwards are destroyed finest first and rebuilt root upwards."""
        assert 1 <= l < len(self.levels)
        for k in range(len(self.links) - 1, l - 2, -1):
            self.links[k].close()
        self.links = self.links[:l - 1]
        self.levels[l] = new_batch
        for k in range(l - 1, len(self.levels) - 1):
            self.links.append(LevelLink(self.levels[k], self.levels[k + 1]))
        self._tables()

    def cfl_dt(self, gamma: float, cfl: float):
        dt, sm = C.c_double(), C.c_double()
        _check(lib().amr_hierarchy_cfl_dt(self._lv, len(self.levels), gamma, cfl, int(self.mhd), C.byref(dt), C.byref(sm)))
        return dt.value, sm.value

    def step(self, dt0: float, gamma: float, limiter: int, riemann: int, ch: float = 0.0, alpha: float = 0.0,
             do_reflux: bool = True):
        _check(lib().amr_hierarchy_step(self._lv, self._lk, len(self.levels), int(self.mhd), dt0, gamma, limiter,
                                        riemann, ch, alpha, int(do_reflux)))

    def close(self):
        for l in reversed(self.links):
            l.close()
        self.links = []

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass


class PatchBuilder:
    """amr_patch_builder: Morton curve order of the leaf cells of a level,
    maximal compact aligned cubic patches, gather into the batch arena layout.  Marshalling only."""

    def __init__(self, ncell_max: int, device: str = "cuda:0", stream: Optional[int] = None):
        import torch  # device memory + stream only
        L = lib()
        nbytes = int(L.amr_builder_bytes(int(ncell_max)))
        if nbytes == 0:
            raise AmrError(-1, "amr_builder_bytes: ncell_max out of range")
        self.device = torch.device(device)
        with torch.cuda.device(self.device):
            self.ws = torch.empty(nbytes, dtype=torch.uint8, device=self.device)
            self.stream = int(torch.cuda.current_stream().cuda_stream) if stream is None else int(stream)
            h = C.c_void_p()
            _check(L.amr_builder_create(int(ncell_max), self.ws.data_ptr(), nbytes, self.stream, C.byref(h)))
        self._h = h
        self.ncell = 0
        self.npatch = 0

    def __del__(self):
        if getattr(self, "_h", None):
            lib().amr_builder_destroy(self._h)
            self._h = None

    def build(self, xyz_dev, bits: int, kmax: int) -> int:
        """xyz_dev: torch int32 CUDA tensor [3, ncell] (contiguous).  Returns the number of patches."""
        assert xyz_dev.is_cuda and xyz_dev.is_contiguous() and xyz_dev.shape[0] == 3
        np_out = C.c_int64(0)
        _check(lib().amr_builder_build(self._h, xyz_dev.data_ptr(), int(xyz_dev.shape[1]), int(bits), int(kmax), C.byref(np_out)))
        self.ncell, self.npatch = int(xyz_dev.shape[1]), int(np_out.value)
        return self.npatch

    def results(self, want_perm: bool = True):
        """(perm [ncell] int64 or None, first [npatch] int64, level [npatch] int32, origin [npatch, 3] int32)."""
        perm = np.empty(self.ncell, np.int64) if want_perm else None
        first = np.empty(self.npatch, np.int64)
        level = np.empty(self.npatch, np.int32)
        origin = np.empty((self.npatch, 3), np.int32)
        _check(lib().amr_builder_results(self._h, perm.ctypes.data if want_perm else None, first.ctypes.data,
                                         level.ctypes.data, origin.ctypes.data))
        return perm, first, level, origin

    def count(self, k: int) -> int:
        c = C.c_int64(0)
        _check(lib().amr_builder_gather(self._h, None, 1, AMR_F32, int(k), None, 0, None, C.byref(c)))
        return int(c.value)

    def gather(self, fields_dev, k: int, want_origin: bool = True):
        """fields_dev: torch CUDA tensor [nf, ncell] float32/float64 in input order.  Returns (out, origin): out a
        torch CUDA tensor [nf, count, n, n, n] (n = 2^k), origin int32 [count, 3] (None and no synchronisation
        with want_origin=False)."""
        import torch
        assert fields_dev.is_cuda and fields_dev.is_contiguous() and fields_dev.shape[1] == self.ncell
        dtype = AMR_F64 if fields_dev.dtype == torch.float64 else AMR_F32
        cnt = self.count(k)
        n = 1 << k
        out = torch.empty((fields_dev.shape[0], cnt, n, n, n), dtype=fields_dev.dtype, device=fields_dev.device)
        origin = np.empty((cnt, 3), np.int32) if want_origin else None
        c = C.c_int64(0)
        _check(lib().amr_builder_gather(self._h, fields_dev.data_ptr(), int(fields_dev.shape[0]), dtype, int(k),
                                        out.data_ptr(), cnt, origin.ctypes.data if want_origin else None, C.byref(c)))
        return out, origin
