"""Thin Python binding over the C-ABI library `libidg_b200.so` (include/idg_b200.h).

Argument marshalling only: every step of the IDG hot path (§2.5 :152-174) runs in the
CUDA kernels behind the C ABI.  PyTorch supplies device memory and streams.  The functions
mirror the C entry points one to one (`idg_grid` -> `grid`, ...).  There is no CPU fallback: if
the library is missing, or a device call is made without a B200, an exception is raised.
"""
from __future__ import annotations

import ctypes
import os
from dataclasses import dataclass

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
# IDG_B200_LIBRARY overrides the in-tree library (used to compare differently compiled builds)
LIB_PATH = os.environ.get("IDG_B200_LIBRARY") or os.path.join(_HERE, "libidg_b200.so")

IDG_GRID, IDG_DEGRID = 0, 1
STAGE_GRIDDER, STAGE_FFT = 0, 1

# every symbol include/idg_b200.h declares
SYMBOLS = (
    "idg_plan_create", "idg_plan_destroy", "idg_plan_counts", "idg_plan_export", "idg_workspace_bytes",
    "idg_grid", "idg_grid_weighted", "idg_degrid", "idg_host_arena_bytes", "idg_host_traffic_bytes", "idg_grid_host", "idg_degrid_host",
    "idg_grid_subgrids", "idg_degrid_subgrids", "idg_subgrid_fft", "idg_adder", "idg_splitter",
    "idg_closure_workspace_bytes", "idg_grid_to_image", "idg_image_to_grid",
    "idg_grid_subgrids_f64", "idg_degrid_subgrids_f64", "idg_power_norm_average",
    "idg_plan_power_norm_terms", "idg_power_norm_average_static",
    "idg_profile_enable", "idg_profile_read", "idg_kernel_config_mask", "idg_plan_kernel_split",
    "idg_measure_alu_peaks", "idg_launch_count", "idg_last_error", "idg_version",
)
KERNEL_KINDS = ("gridder", "fft", "adder", "splitter", "ifft", "degridder")


class IdgError(RuntimeError):
    pass


class _Params(ctypes.Structure):
    _fields_ = [
        ("grid_size", ctypes.c_int32), ("subgrid_size", ctypes.c_int32), ("padding", ctypes.c_int32),
        ("n_stations", ctypes.c_int32), ("n_baselines", ctypes.c_int32), ("n_times", ctypes.c_int32),
        ("n_chan", ctypes.c_int32), ("aterm_period", ctypes.c_int32),
        ("cell_size", ctypes.c_double), ("w_step", ctypes.c_double), ("comfort", ctypes.c_double),
        ("max_batch_subgrids", ctypes.c_int64),
        ("gridder_variant", ctypes.c_int32), ("degridder_variant", ctypes.c_int32),
        ("positive_w", ctypes.c_int32), ("power_norm", ctypes.c_int32),
    ]


_lib = None


def load_library() -> ctypes.CDLL:
    """dlopen the in-tree library; raises if it has not been built (see build.py)."""
    global _lib
    if _lib is not None:
        return _lib
    if not os.path.exists(LIB_PATH):
        raise IdgError(f"{LIB_PATH} not found: build it with `python -m paper_2502_17789_b200.build` "
                       "(there is no CPU fallback)")
    lib = ctypes.CDLL(LIB_PATH)
    vp, i64, i32, sz = ctypes.c_void_p, ctypes.c_int64, ctypes.c_int32, ctypes.c_size_t
    lib.idg_plan_create.argtypes = [ctypes.POINTER(_Params), vp, vp, vp, ctypes.POINTER(vp)]
    lib.idg_plan_create.restype = ctypes.c_int
    lib.idg_plan_destroy.argtypes = [vp]
    lib.idg_plan_destroy.restype = None
    lib.idg_plan_counts.argtypes = [vp, ctypes.POINTER(i64), ctypes.POINTER(i32), ctypes.POINTER(i32),
                                    ctypes.POINTER(i64), ctypes.POINTER(i64)]
    lib.idg_plan_counts.restype = ctypes.c_int
    lib.idg_plan_export.argtypes = [vp, vp]
    lib.idg_plan_export.restype = ctypes.c_int
    lib.idg_workspace_bytes.argtypes = [vp, ctypes.c_int]
    lib.idg_workspace_bytes.restype = sz
    lib.idg_host_arena_bytes.argtypes = [vp, ctypes.c_int]
    lib.idg_host_arena_bytes.restype = sz
    lib.idg_host_traffic_bytes.argtypes = [vp, ctypes.c_int, ctypes.POINTER(i64), ctypes.POINTER(i64)]
    lib.idg_host_traffic_bytes.restype = ctypes.c_int
    lib.idg_grid.argtypes = [vp, vp, vp, vp, vp, vp, sz, vp]
    lib.idg_grid.restype = ctypes.c_int
    lib.idg_grid_weighted.argtypes = [vp, vp, vp, vp, vp, vp, vp, sz, vp]
    lib.idg_grid_weighted.restype = ctypes.c_int
    lib.idg_degrid.argtypes = [vp, vp, vp, vp, vp, vp, sz, vp]
    lib.idg_degrid.restype = ctypes.c_int
    lib.idg_grid_host.argtypes = [vp, vp, vp, vp, vp, vp, sz, vp]
    lib.idg_grid_host.restype = ctypes.c_int
    lib.idg_degrid_host.argtypes = [vp, vp, vp, vp, vp, vp, sz, vp]
    lib.idg_degrid_host.restype = ctypes.c_int
    lib.idg_grid_subgrids.argtypes = [vp, i64, i64, vp, vp, vp, vp, ctypes.c_int, vp]
    lib.idg_grid_subgrids.restype = ctypes.c_int
    lib.idg_degrid_subgrids.argtypes = [vp, i64, i64, vp, vp, vp, vp, vp]
    lib.idg_degrid_subgrids.restype = ctypes.c_int
    lib.idg_subgrid_fft.argtypes = [i32, i64, vp, ctypes.c_int, vp]
    lib.idg_subgrid_fft.restype = ctypes.c_int
    lib.idg_adder.argtypes = [vp, i64, i64, vp, vp, vp]
    lib.idg_adder.restype = ctypes.c_int
    lib.idg_splitter.argtypes = [vp, i64, i64, vp, vp, vp]
    lib.idg_splitter.restype = ctypes.c_int
    lib.idg_closure_workspace_bytes.argtypes = [vp]
    lib.idg_closure_workspace_bytes.restype = sz
    lib.idg_grid_to_image.argtypes = [vp, vp, vp, vp, vp, sz, vp]
    lib.idg_grid_to_image.restype = ctypes.c_int
    lib.idg_image_to_grid.argtypes = [vp, vp, vp, vp, vp]
    lib.idg_image_to_grid.restype = ctypes.c_int
    lib.idg_profile_enable.argtypes = [ctypes.c_int]
    lib.idg_profile_enable.restype = ctypes.c_int
    lib.idg_profile_read.argtypes = [vp, vp]
    lib.idg_profile_read.restype = ctypes.c_int
    lib.idg_plan_kernel_split.argtypes = [vp, ctypes.c_int, ctypes.POINTER(i64), ctypes.POINTER(i64)]
    lib.idg_plan_kernel_split.restype = ctypes.c_int
    lib.idg_kernel_config_mask.argtypes = [ctypes.c_int, ctypes.c_int]
    lib.idg_kernel_config_mask.restype = ctypes.c_int
    lib.idg_grid_subgrids_f64.argtypes = [vp, i64, i64, vp, vp, vp, vp, vp]
    lib.idg_grid_subgrids_f64.restype = ctypes.c_int
    lib.idg_degrid_subgrids_f64.argtypes = [vp, i64, i64, vp, vp, vp, vp, vp]
    lib.idg_degrid_subgrids_f64.restype = ctypes.c_int
    lib.idg_power_norm_average.argtypes = [vp, vp, vp, vp]
    lib.idg_power_norm_average.restype = ctypes.c_int
    lib.idg_plan_power_norm_terms.argtypes = [vp, vp, vp, i64, ctypes.POINTER(i64), ctypes.POINTER(ctypes.c_double)]
    lib.idg_plan_power_norm_terms.restype = ctypes.c_int
    lib.idg_power_norm_average_static.argtypes = [vp, ctypes.c_int32, ctypes.c_int32, vp, vp, i64, ctypes.c_double, vp, vp]
    lib.idg_power_norm_average_static.restype = ctypes.c_int
    lib.idg_measure_alu_peaks.argtypes = [vp]
    lib.idg_measure_alu_peaks.restype = ctypes.c_int
    lib.idg_launch_count.argtypes = []
    lib.idg_launch_count.restype = i64
    lib.idg_last_error.argtypes = []
    lib.idg_last_error.restype = ctypes.c_char_p
    lib.idg_version.argtypes = []
    lib.idg_version.restype = ctypes.c_char_p
    _lib = lib
    return lib


def _check(rc: int, what: str) -> None:
    if rc != 0:
        msg = load_library().idg_last_error().decode("utf-8", "replace")
        raise IdgError(f"{what} failed with code {rc}: {msg}")


def _ptr(t) -> int:
    """Device / host pointer of a torch tensor or numpy array (contiguous)."""
    if isinstance(t, np.ndarray):
        if not t.flags["C_CONTIGUOUS"]:
            raise ValueError("array must be C-contiguous")
        return t.ctypes.data
    if not t.is_contiguous():
        raise ValueError("tensor must be contiguous")
    return t.data_ptr()


def _stream_ptr(stream) -> int | None:
    if stream is None:
        import torch
        return torch.cuda.current_stream().cuda_stream
    return stream.cuda_stream if hasattr(stream, "cuda_stream") else int(stream)


def _need_cuda(*tensors) -> None:
    for t in tensors:
        if not getattr(t, "is_cuda", False):
            raise IdgError("device entry points need CUDA tensors (there is no CPU fallback)")


@dataclass(frozen=True)
class PlanCounts:
    n_subgrids: int
    n_wlayers: int
    wl_min: int
    n_vis_planned: int
    n_vis_dropped: int


VARIANT_AUTO, VARIANT_SIMT, VARIANT_TENSOR, VARIANT_FP64 = 0, 1, 2, 3
KMASK_SIMT, KMASK_FP64, KMASK_ROT = 1 << 0, 1 << 8, 1 << 9


def kmask_tc(ng: int) -> int:
    """Bit of idg_kernel_config_mask for the tensor-core kernel with `ng` compute groups per CTA."""
    return 1 << ng


class Plan:
    """Owner of an `idg_plan*` (idg_plan_create / idg_plan_destroy)."""

    def __init__(self, *, grid_size, subgrid_size, padding, cell_size, w_step, n_stations, n_times, n_chan,
                 aterm_period, uvw_m, freqs, baselines, comfort=0.75, max_batch_subgrids=0,
                 gridder_variant=VARIANT_AUTO, degridder_variant=VARIANT_AUTO, positive_w=False, power_norm=False):
        lib = load_library()
        uvw_m = np.ascontiguousarray(uvw_m, dtype=np.float64)
        freqs = np.ascontiguousarray(freqs, dtype=np.float64)
        baselines = np.ascontiguousarray(baselines, dtype=np.int32)
        n_bl = baselines.shape[0]
        if uvw_m.shape != (n_bl * n_times, 3) or freqs.shape != (n_chan,) or baselines.shape != (n_bl, 2):
            raise ValueError("uvw_m must be [n_bl*n_times,3], freqs [n_chan], baselines [n_bl,2]")
        self.params = _Params(grid_size, subgrid_size, padding, n_stations, n_bl, n_times, n_chan, aterm_period,
                              cell_size, w_step, comfort, max_batch_subgrids, int(gridder_variant),
                              int(degridder_variant), int(bool(positive_w)), int(bool(power_norm)))
        handle = ctypes.c_void_p()
        _check(lib.idg_plan_create(ctypes.byref(self.params), uvw_m.ctypes.data, freqs.ctypes.data,
                                   baselines.ctypes.data, ctypes.byref(handle)), "idg_plan_create")
        self._h = handle
        self.n_rows = n_bl * n_times
        self.n_chan = n_chan
        self.n_stations = n_stations
        self.subgrid_size = subgrid_size
        self.grid_size = grid_size
        self.n_intervals = -(-n_times // aterm_period)
        self._counts = None

    def __del__(self):
        h = getattr(self, "_h", None)
        if h and _lib is not None:
            _lib.idg_plan_destroy(h)
            self._h = None

    @property
    def handle(self):
        return self._h

    def counts(self) -> PlanCounts:
        if self._counts is None:
            n, w, wl, pl, dr = (ctypes.c_int64(), ctypes.c_int32(), ctypes.c_int32(), ctypes.c_int64(),
                                ctypes.c_int64())
            _check(load_library().idg_plan_counts(self._h, ctypes.byref(n), ctypes.byref(w), ctypes.byref(wl),
                                                  ctypes.byref(pl), ctypes.byref(dr)), "idg_plan_counts")
            self._counts = PlanCounts(n.value, w.value, wl.value, pl.value, dr.value)
        return self._counts

    def export(self) -> np.ndarray:
        n = self.counts().n_subgrids
        sub = np.zeros((n, 8), np.int32)
        _check(load_library().idg_plan_export(self._h, sub.ctypes.data), "idg_plan_export")
        return sub

    def workspace_bytes(self, direction=IDG_GRID) -> int:
        return int(load_library().idg_workspace_bytes(self._h, direction))

    def host_arena_bytes(self, direction=IDG_GRID) -> int:
        return int(load_library().idg_host_arena_bytes(self._h, direction))

    def host_traffic_bytes(self, direction=IDG_GRID):
        """(host-to-device, device-to-host) bytes of one grid_host / degrid_host call."""
        up, down = ctypes.c_int64(), ctypes.c_int64()
        _check(load_library().idg_host_traffic_bytes(self._h, direction, ctypes.byref(up), ctypes.byref(down)),
               "idg_host_traffic_bytes")
        return int(up.value), int(down.value)

    def kernel_split(self, direction=IDG_GRID):
        """(tensor-core, SIMT) subgrid counts of a direction under the plan's kernel variant."""
        nt, ns = ctypes.c_int64(), ctypes.c_int64()
        _check(load_library().idg_plan_kernel_split(self._h, direction, ctypes.byref(nt), ctypes.byref(ns)),
               "idg_plan_kernel_split")
        return int(nt.value), int(ns.value)

    def closure_workspace_bytes(self) -> int:
        return int(load_library().idg_closure_workspace_bytes(self._h))

    # ---- sizes of the arrays the C ABI takes (it sees only pointers: the binding checks dtype and size)
    def vis_numel(self) -> int:
        return self.n_rows * self.n_chan * 4

    def aterms_numel(self) -> int:
        L = self.subgrid_size
        return self.n_stations * self.n_intervals * L * L * 4

    def grid_numel(self) -> int:
        return self.counts().n_wlayers * 4 * self.grid_size * self.grid_size


def plan_from_config(cfg, uvw_m, freqs, baselines, max_batch_subgrids=0, **kw) -> Plan:
    """Convenience: a Plan from a `synth.Config`-like object (attribute names as in include/idg_b200.h);
    kw: gridder_variant, degridder_variant, positive_w, power_norm."""
    return Plan(grid_size=cfg.grid_size, subgrid_size=cfg.subgrid_size, padding=cfg.padding,
                cell_size=cfg.cell_size, w_step=cfg.w_step, n_stations=cfg.n_stations, n_times=cfg.n_times,
                n_chan=cfg.n_chan, aterm_period=cfg.aterm_period, uvw_m=uvw_m, freqs=freqs, baselines=baselines,
                comfort=cfg.comfort, max_batch_subgrids=max_batch_subgrids, **kw)


_DTYPES = {"c64": ("complex64",), "c128": ("complex128",), "f32": ("float32",), "f64": ("float64",), "i32": ("int32",)}


def _expect(t, kind: str, numel: int, what: str, at_least: bool = False) -> None:
    """dtype and element count of an array handed to the C ABI (which cannot see either); `at_least` for
    buffers of which a call may use only the leading part."""
    name = str(t.dtype).replace("torch.", "")
    if name not in _DTYPES[kind]:
        raise ValueError(f"{what}: dtype {name}, expected {_DTYPES[kind][0]}")
    n = int(t.numel()) if hasattr(t, "numel") else int(t.size)
    if n != numel and not (at_least and n > numel):
        raise ValueError(f"{what}: {n} elements, expected {numel}")


def _expect_common(plan: Plan, vis=None, aterms=None, taper=None, grid=None, vis_kind="c64") -> None:
    L = plan.subgrid_size
    if vis is not None:
        _expect(vis, vis_kind, plan.vis_numel(), "vis [n_rows, n_chan, 4]")
    if aterms is not None:
        _expect(aterms, "c64", plan.aterms_numel(), "aterms [n_stations, n_intervals, L, L, 2, 2]")
    if taper is not None:
        _expect(taper, "f32", L * L, "taper [L, L]")
    if grid is not None:
        _expect(grid, "c64", plan.grid_numel(), "grid [n_wlayers, 4, Ng, Ng]")


def _nbytes(t) -> int:
    return t.numel() * t.element_size()


def grid(plan: Plan, vis, aterms, taper, grid_out, workspace, stream=None) -> None:
    """idg_grid: accumulate all subgrids of the plan into grid_out [W,4,Ng,Ng] complex64."""
    _need_cuda(vis, aterms, taper, grid_out, workspace)
    _expect_common(plan, vis, aterms, taper, grid_out)
    _check(load_library().idg_grid(plan.handle, _ptr(vis), _ptr(aterms), _ptr(taper), _ptr(grid_out),
                                   _ptr(workspace), _nbytes(workspace), _stream_ptr(stream)), "idg_grid")


def grid_weighted(plan: Plan, vis, weights, aterms, taper, grid_out, workspace, stream=None) -> None:
    """idg_grid_weighted: as grid(), with vis[r, c, :] * weights[r, c] (float32) applied at load."""
    _need_cuda(vis, weights, aterms, taper, grid_out, workspace)
    _expect_common(plan, vis, aterms, taper, grid_out)
    _expect(weights, "f32", plan.n_rows * plan.n_chan, "weights [n_rows, n_chan]")
    _check(load_library().idg_grid_weighted(plan.handle, _ptr(vis), _ptr(weights), _ptr(aterms), _ptr(taper),
                                            _ptr(grid_out), _ptr(workspace), _nbytes(workspace),
                                            _stream_ptr(stream)), "idg_grid_weighted")


def grid_to_image(plan: Plan, grid_in, image_out, workspace, corr=None, stream=None) -> None:
    """idg_grid_to_image (w-stacking closure, outside the hot path): image_out [4,Ng,Ng] complex64."""
    _need_cuda(grid_in, image_out, workspace, *(() if corr is None else (corr,)))
    _expect_common(plan, grid=grid_in)
    _expect(image_out, "c64", 4 * plan.grid_size ** 2, "image [4, Ng, Ng]")
    if corr is not None:
        _expect(corr, "f32", plan.grid_size ** 2, "corr [Ng, Ng]")
    _check(load_library().idg_grid_to_image(plan.handle, _ptr(grid_in), None if corr is None else _ptr(corr),
                                            _ptr(image_out), _ptr(workspace), _nbytes(workspace),
                                            _stream_ptr(stream)), "idg_grid_to_image")


def image_to_grid(plan: Plan, image_in, grid_out, corr=None, stream=None) -> None:
    """idg_image_to_grid: grid_out [W,4,Ng,Ng] complex64 is overwritten."""
    _need_cuda(image_in, grid_out, *(() if corr is None else (corr,)))
    _expect_common(plan, grid=grid_out)
    _expect(image_in, "c64", 4 * plan.grid_size ** 2, "image [4, Ng, Ng]")
    if corr is not None:
        _expect(corr, "f32", plan.grid_size ** 2, "corr [Ng, Ng]")
    _check(load_library().idg_image_to_grid(plan.handle, _ptr(image_in), None if corr is None else _ptr(corr),
                                            _ptr(grid_out), _stream_ptr(stream)), "idg_image_to_grid")


def degrid(plan: Plan, grid_in, aterms, taper, vis_out, workspace, stream=None) -> None:
    """idg_degrid: predict every planned visibility into vis_out [n_rows,n_chan,4] complex64."""
    _need_cuda(vis_out, aterms, taper, grid_in, workspace)
    _expect_common(plan, vis_out, aterms, taper, grid_in)
    _check(load_library().idg_degrid(plan.handle, _ptr(grid_in), _ptr(aterms), _ptr(taper), _ptr(vis_out),
                                     _ptr(workspace), _nbytes(workspace), _stream_ptr(stream)), "idg_degrid")


def grid_host(plan: Plan, vis, aterms, taper, grid_io, arena, stream=None) -> None:
    """idg_grid_host: host buffers in, host grid accumulated; copies run inside the call."""
    _need_cuda(arena)
    _expect_common(plan, vis, aterms, taper, grid_io)
    _check(load_library().idg_grid_host(plan.handle, _ptr(vis), _ptr(aterms), _ptr(taper), _ptr(grid_io),
                                        _ptr(arena), _nbytes(arena), _stream_ptr(stream)), "idg_grid_host")


def degrid_host(plan: Plan, grid_in, aterms, taper, vis_io, arena, stream=None) -> None:
    """idg_degrid_host: host buffers in, host visibilities out."""
    _need_cuda(arena)
    _expect_common(plan, vis_io, aterms, taper, grid_in)
    _check(load_library().idg_degrid_host(plan.handle, _ptr(grid_in), _ptr(aterms), _ptr(taper), _ptr(vis_io),
                                          _ptr(arena), _nbytes(arena), _stream_ptr(stream)), "idg_degrid_host")


def grid_subgrids(plan: Plan, first, count, vis, aterms, taper, subgrids_out, stage=STAGE_FFT, stream=None) -> None:
    _need_cuda(vis, aterms, taper, subgrids_out)
    _expect_common(plan, vis, aterms, taper)
    _expect(subgrids_out, "c64", count * 4 * plan.subgrid_size ** 2, "subgrids [count, 4, L, L]", at_least=True)
    _check(load_library().idg_grid_subgrids(plan.handle, first, count, _ptr(vis), _ptr(aterms), _ptr(taper),
                                            _ptr(subgrids_out), stage, _stream_ptr(stream)), "idg_grid_subgrids")


def degrid_subgrids(plan: Plan, first, count, subgrids_in, aterms, taper, vis_out, stream=None) -> None:
    _need_cuda(vis_out, aterms, taper, subgrids_in)
    _expect_common(plan, vis_out, aterms, taper)
    _expect(subgrids_in, "c64", count * 4 * plan.subgrid_size ** 2, "subgrids [count, 4, L, L]", at_least=True)
    _check(load_library().idg_degrid_subgrids(plan.handle, first, count, _ptr(subgrids_in), _ptr(aterms),
                                              _ptr(taper), _ptr(vis_out), _stream_ptr(stream)),
           "idg_degrid_subgrids")


def grid_subgrids_f64(plan: Plan, first, count, vis, aterms, taper, subgrids_out, stream=None) -> None:
    """idg_grid_subgrids_f64: the fp64 gridder + A-term / taper; subgrids_out [count,4,L,L] complex128."""
    _need_cuda(vis, aterms, taper, subgrids_out)
    _expect_common(plan, vis, aterms, taper)
    _expect(subgrids_out, "c128", count * 4 * plan.subgrid_size ** 2, "subgrids [count, 4, L, L]", at_least=True)
    _check(load_library().idg_grid_subgrids_f64(plan.handle, first, count, _ptr(vis), _ptr(aterms), _ptr(taper),
                                                _ptr(subgrids_out), _stream_ptr(stream)), "idg_grid_subgrids_f64")


def degrid_subgrids_f64(plan: Plan, first, count, subgrids_in, aterms, taper, vis_out, stream=None) -> None:
    """idg_degrid_subgrids_f64: complex128 subgrids in, complex128 visibilities out."""
    _need_cuda(vis_out, aterms, taper, subgrids_in)
    _expect_common(plan, vis_out, aterms, taper, vis_kind="c128")
    _expect(subgrids_in, "c128", count * 4 * plan.subgrid_size ** 2, "subgrids [count, 4, L, L]", at_least=True)
    _check(load_library().idg_degrid_subgrids_f64(plan.handle, first, count, _ptr(subgrids_in), _ptr(aterms),
                                                  _ptr(taper), _ptr(vis_out), _stream_ptr(stream)),
           "idg_degrid_subgrids_f64")


def power_norm_average(plan: Plan, aterms, avg_out, stream=None) -> None:
    """idg_power_norm_average: avg_out [L, L] float64, the visibility-weighted mean of 1 / ||M_p M_q^H||_F."""
    _need_cuda(aterms, avg_out)
    _expect_common(plan, aterms=aterms)
    _expect(avg_out, "f64", plan.subgrid_size ** 2, "avg [L, L]")
    _check(load_library().idg_power_norm_average(plan.handle, _ptr(aterms), _ptr(avg_out), _stream_ptr(stream)),
           "idg_power_norm_average")


def plan_power_norm_terms(plan: Plan):
    """idg_plan_power_norm_terms (host only): (pairs [n, 3] int32 of (p, q, interval), weights [n] float64,
    weight_sum) -- the inputs of power_norm_average_static, in the order idg_power_norm_average uses."""
    lib = load_library()
    n, wsum = ctypes.c_int64(0), ctypes.c_double(0.0)
    _check(lib.idg_plan_power_norm_terms(plan.handle, None, None, 0, ctypes.byref(n), ctypes.byref(wsum)),
           "idg_plan_power_norm_terms")
    pairs = np.zeros((n.value, 3), np.int32)
    weights = np.zeros(n.value, np.float64)
    if n.value:
        _check(lib.idg_plan_power_norm_terms(plan.handle, pairs.ctypes.data, weights.ctypes.data, n.value,
                                             ctypes.byref(n), ctypes.byref(wsum)), "idg_plan_power_norm_terms")
    return pairs, weights, float(wsum.value)


def power_norm_average_static(aterms, subgrid_size, n_intervals, pairs, weights, weight_sum, avg_out,
                              stream=None) -> None:
    """idg_power_norm_average_static: the average of power_norm_average without any device allocation (scratch
    built into the library, subgrid_size <= 96, calls on one device must not overlap).  Every array is a CUDA
    tensor the caller owns: pairs [n, 3] int32, weights [n] float64, avg_out [L, L] float64."""
    _need_cuda(aterms, pairs, weights, avg_out)
    n = int(weights.numel())
    _expect(pairs, "i32", n * 3, "pairs [n_terms, 3]")
    _expect(weights, "f64", n, "weights [n_terms]")
    _expect(avg_out, "f64", subgrid_size ** 2, "avg [L, L]")
    _check(load_library().idg_power_norm_average_static(_ptr(aterms), int(subgrid_size), int(n_intervals), _ptr(pairs),
                                                        _ptr(weights), n, float(weight_sum), _ptr(avg_out),
                                                        _stream_ptr(stream)), "idg_power_norm_average_static")


def subgrid_fft(subgrid_size, planes, direction, stream=None) -> None:
    """idg_subgrid_fft: planes [..., L, L] complex64, transformed in place."""
    _need_cuda(planes)
    n_planes = planes.numel() // (subgrid_size * subgrid_size)
    _expect(planes, "c64", n_planes * subgrid_size * subgrid_size, "planes [..., L, L]")
    _check(load_library().idg_subgrid_fft(subgrid_size, n_planes, _ptr(planes), direction, _stream_ptr(stream)),
           "idg_subgrid_fft")


def adder(plan: Plan, first, count, subgrids, grid_io, stream=None) -> None:
    _need_cuda(subgrids, grid_io)
    _expect_common(plan, grid=grid_io)
    _expect(subgrids, "c64", count * 4 * plan.subgrid_size ** 2, "subgrids [count, 4, L, L]", at_least=True)
    _check(load_library().idg_adder(plan.handle, first, count, _ptr(subgrids), _ptr(grid_io), _stream_ptr(stream)),
           "idg_adder")


def splitter(plan: Plan, first, count, grid_in, subgrids_out, stream=None) -> None:
    _need_cuda(subgrids_out, grid_in)
    _expect_common(plan, grid=grid_in)
    _expect(subgrids_out, "c64", count * 4 * plan.subgrid_size ** 2, "subgrids [count, 4, L, L]", at_least=True)
    _check(load_library().idg_splitter(plan.handle, first, count, _ptr(grid_in), _ptr(subgrids_out),
                                       _stream_ptr(stream)), "idg_splitter")


def profile_enable(on: bool) -> None:
    _check(load_library().idg_profile_enable(1 if on else 0), "idg_profile_enable")


def profile_read() -> dict:
    """idg_profile_read: {kind: (milliseconds, launches)} accumulated since the last read."""
    ms = np.zeros(len(KERNEL_KINDS), np.float64)
    n = np.zeros(len(KERNEL_KINDS), np.int64)
    _check(load_library().idg_profile_read(ms.ctypes.data, n.ctypes.data), "idg_profile_read")
    return {k: (float(ms[i]), int(n[i])) for i, k in enumerate(KERNEL_KINDS)}


def kernel_config_mask(kind: str, reset: bool = False) -> int:
    """idg_kernel_config_mask: which kernels the direct-sum step `kind` ("gridder" | "degridder") launched."""
    m = int(load_library().idg_kernel_config_mask(KERNEL_KINDS.index(kind), 1 if reset else 0))
    if m < 0:
        _check(m, "idg_kernel_config_mask")
    return m


def measure_alu_peaks() -> dict:
    """idg_measure_alu_peaks: empirical per-SM-per-clock rates of the FP32 and SFU pipes."""
    out = np.zeros(7, np.float64)
    _check(load_library().idg_measure_alu_peaks(out.ctypes.data), "idg_measure_alu_peaks")
    return dict(ffma=float(out[0]), ffma2=float(out[1]), mufu_ex2=float(out[2]), sincos=float(out[3]),
                gridder_mix_pairs=float(out[4]), gridder_mix_scalar_pairs=float(out[5]),
                operand_gen_pairs=float(out[6]))


def launch_count() -> int:
    return int(load_library().idg_launch_count())


def version() -> str:
    return load_library().idg_version().decode()
