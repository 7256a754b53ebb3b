"""ctypes binding of include/phylino.h.  Argument marshalling only.

PyTorch is used for what the caller hands in and gets back (device tensors, the current CUDA
stream); nothing here computes.
"""
from __future__ import annotations

import ctypes as C
import os
from typing import Optional, Sequence

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
# PHYLINO_LIBRARY: another build of the same library (e.g. libphylino_checked.so, python -m ...build --checked)
_LIB_PATH = os.environ.get("PHYLINO_LIBRARY") or os.path.join(_HERE, "libphylino.so")

# every symbol include/phylino.h declares
abi_symbols = (
    "phylino_create", "phylino_destroy", "phylino_set_model", "phylino_load_events",
    "phylino_spectra", "phylino_nll", "phylino_event_bins", "phylino_nll_host",
    "phylino_spectra_host", "phylino_total_bins", "phylino_total_events",
    "phylino_set_tuning", "phylino_launch_count", "phylino_last_error", "phylino_peak_fp64",
    "phylino_expectation", "phylino_set_timing", "phylino_last_kernel_ms",
    "phylino_set_caching", "phylino_last_plan", "phylino_set_prior_blocks",
    "phylino_nll_ensemble", "phylino_set_transform", "phylino_param_width",
    "phylino_launch_floor", "phylino_set_schedule", "phylino_reserve",
    "phylino_draw_pseudo_data", "phylino_ordering_scan", "phylino_nll_gradient",
    "phylino_set_energy_correction_mode", "phylino_set_flux_model", "phylino_last_small_phase",
    "phylino_hbm_read_floor", "phylino_last_medium_phase", "phylino_set_functions",
    "phylino_variable_metric_step", "phylino_variable_metric_step_static",
)

_STATUS = {0: "OK", 1: "ERR_ARG", 2: "ERR_SHAPE", 3: "ERR_STATE", 4: "ERR_OOM", 5: "ERR_CUDA"}


class PhylinoError(RuntimeError):
    def __init__(self, status: int, text: str):
        super().__init__(f"phylino: {_STATUS.get(status, status)}: {text}")
        self.status = status


class _Bkg(C.Structure):
    _fields_ = [("idx_rate", C.c_int32), ("tmpl", C.c_void_p), ("idx_shape", C.c_void_p)]


class _Dataset(C.Structure):
    _fields_ = [("n_bins", C.c_int32), ("idx_a", C.c_int32 * 3), ("idx_signorm", C.c_int32),
                ("norm", C.c_double), ("idx_flux", C.c_void_p), ("n_bkg", C.c_int32),
                ("bkg", C.POINTER(_Bkg))]


class _PriorBlock(C.Structure):
    _fields_ = [("n", C.c_int32), ("idx", C.c_void_p), ("mean", C.c_void_p), ("inv_cov", C.c_void_p)]


class _Monomial(C.Structure):
    _fields_ = [("coef", C.c_double), ("n_factors", C.c_int32), ("idx", C.c_void_p), ("power", C.c_void_p)]


class _Function(C.Structure):
    _fields_ = [("offset", C.c_double), ("n_terms", C.c_int32), ("terms", C.POINTER(_Monomial))]


class _TransformBlock(C.Structure):
    _fields_ = [("n_out", C.c_int32), ("n_in", C.c_int32), ("idx_out", C.c_void_p), ("idx_in", C.c_void_p),
                ("offset", C.c_void_p), ("centre", C.c_void_p), ("matrix", C.c_void_p)]


class _Model(C.Structure):
    _fields_ = [("osc_model", C.c_int32), ("ordering", C.c_int32), ("n_params", C.c_int32),
                ("n_datasets", C.c_int32), ("idx_osc", C.c_int32 * 6), ("fixed_osc", C.c_double * 6),
                ("datasets", C.POINTER(_Dataset)), ("prior_mean", C.c_void_p),
                ("prior_sigma", C.c_void_p)]


_lib = None


def lib_path() -> str:
    return _LIB_PATH


def load_library():
    """dlopen libphylino.so.  Fails loudly if it has not been built (no fallback of any kind)."""
    global _lib
    if _lib is not None:
        return _lib
    if not os.path.exists(_LIB_PATH):
        raise RuntimeError(
            f"{_LIB_PATH} is missing: build it with `python -m paper_2502_15253_b200.build` "
            "(nvcc, sm_100a).  There is no CPU or PyTorch fallback for this path.")
    lib = C.CDLL(_LIB_PATH)
    vp, i32, i64, dbl = C.c_void_p, C.c_int, C.c_int64, C.c_double
    lib.phylino_create.restype = i32
    lib.phylino_create.argtypes = [i32, vp, C.POINTER(vp)]
    lib.phylino_destroy.restype = None
    lib.phylino_destroy.argtypes = [vp]
    lib.phylino_set_model.restype = i32
    lib.phylino_set_model.argtypes = [vp, C.POINTER(_Model)]
    lib.phylino_load_events.restype = i32
    lib.phylino_load_events.argtypes = [vp, i32, i64, vp, vp, vp, vp, i32, vp, i32, vp]
    lib.phylino_spectra.restype = i32
    lib.phylino_spectra.argtypes = [vp, i32, vp, vp]
    lib.phylino_nll.restype = i32
    lib.phylino_nll.argtypes = [vp, i32, vp, vp, vp]
    lib.phylino_expectation.restype = i32
    lib.phylino_expectation.argtypes = [vp, i32, vp, vp]
    lib.phylino_set_timing.restype = i32
    lib.phylino_set_timing.argtypes = [vp, i32]
    lib.phylino_last_kernel_ms.restype = i32
    lib.phylino_last_kernel_ms.argtypes = [vp, C.POINTER(C.c_float)]
    lib.phylino_event_bins.restype = i32
    lib.phylino_event_bins.argtypes = [vp, i32, vp, vp]
    lib.phylino_nll_host.restype = i32
    lib.phylino_nll_host.argtypes = [vp, i32, vp, vp, vp]
    lib.phylino_spectra_host.restype = i32
    lib.phylino_spectra_host.argtypes = [vp, i32, vp, vp]
    lib.phylino_total_bins.restype = i64
    lib.phylino_total_bins.argtypes = [vp]
    lib.phylino_total_events.restype = i64
    lib.phylino_total_events.argtypes = [vp]
    lib.phylino_set_transform.restype = i32
    lib.phylino_set_transform.argtypes = [vp, i32, vp, vp, i32, C.POINTER(_TransformBlock)]
    lib.phylino_param_width.restype = i64
    lib.phylino_param_width.argtypes = [vp]
    lib.phylino_nll_ensemble.restype = i32
    lib.phylino_nll_ensemble.argtypes = [vp, i32, vp, i32, vp, vp]
    lib.phylino_set_prior_blocks.restype = i32
    lib.phylino_set_prior_blocks.argtypes = [vp, i32, C.POINTER(_PriorBlock)]
    lib.phylino_variable_metric_step.restype = i32
    lib.phylino_variable_metric_step.argtypes = [vp, i32, vp, vp, vp, vp, vp, vp]
    lib.phylino_variable_metric_step_static.restype = i32
    lib.phylino_variable_metric_step_static.argtypes = [vp, i32, vp, vp, vp, vp, vp, vp, C.c_char_p, i32]
    lib.phylino_set_functions.restype = i32
    lib.phylino_set_functions.argtypes = [vp, i32, C.POINTER(_Function)]
    lib.phylino_set_caching.restype = i32
    lib.phylino_set_caching.argtypes = [vp, i32]
    lib.phylino_last_plan.restype = i32
    lib.phylino_last_plan.argtypes = [vp, C.POINTER(C.c_int64), C.POINTER(C.c_int64)]
    lib.phylino_set_tuning.restype = i32
    lib.phylino_set_tuning.argtypes = [vp, i32, i32, i32]
    lib.phylino_draw_pseudo_data.restype = i32
    lib.phylino_draw_pseudo_data.argtypes = [vp, vp, i32, C.c_uint64, vp]
    lib.phylino_ordering_scan.restype = i32
    lib.phylino_ordering_scan.argtypes = [vp, i32, i32, vp, vp, vp, vp]
    lib.phylino_nll_gradient.restype = i32
    lib.phylino_nll_gradient.argtypes = [vp, vp, vp, vp, vp, vp]
    lib.phylino_set_energy_correction_mode.restype = i32
    lib.phylino_set_energy_correction_mode.argtypes = [vp, i32]
    lib.phylino_set_flux_model.restype = i32
    lib.phylino_set_flux_model.argtypes = [vp, i32, i32, vp, dbl, dbl]
    lib.phylino_last_small_phase.restype = i32
    lib.phylino_last_small_phase.argtypes = [vp, C.POINTER(dbl)]
    lib.phylino_last_medium_phase.restype = i32
    lib.phylino_last_medium_phase.argtypes = [vp, C.POINTER(dbl)]
    lib.phylino_set_schedule.restype = i32
    lib.phylino_set_schedule.argtypes = [vp, i32]
    lib.phylino_reserve.restype = i32
    lib.phylino_reserve.argtypes = [vp, i32]
    lib.phylino_launch_count.restype = i64
    lib.phylino_launch_count.argtypes = [vp]
    lib.phylino_last_error.restype = C.c_char_p
    lib.phylino_last_error.argtypes = [vp]
    lib.phylino_launch_floor.restype = i32
    lib.phylino_launch_floor.argtypes = [vp, i32, C.POINTER(dbl)]
    lib.phylino_hbm_read_floor.restype = i32
    lib.phylino_hbm_read_floor.argtypes = [vp, i64, i32, C.POINTER(dbl)]
    lib.phylino_peak_fp64.restype = i32
    lib.phylino_peak_fp64.argtypes = [vp, i32, C.POINTER(dbl)]
    _lib = lib
    return lib


def _np_ptr(a: Optional[np.ndarray]):
    return None if a is None else a.ctypes.data


STATIC_MAX_N = 2048      # PHYLINO_STATIC_MAX_N


def variable_metric_step_static(V, grad, dx=None, dg=None, direction=None, edm=None, stream: Optional[int] = None):
    """phylino_variable_metric_step_static: the variable-metric step without a context and without any device
    allocation by the library -- for callers whose GPU memory belongs to another allocator, who cannot take the
    device-wide stall of a cudaMalloc, or who may not allocate after start-up.  The library's scratch is a fixed
    array (N <= STATIC_MAX_N) shared by all calls on a device: keep them on one stream.

    V [N, N] float64 CUDA, updated IN PLACE from the last move dx and gradient change dg (both or neither).  Pass
    preallocated `direction` [N] and `edm` [2] to keep this wrapper from allocating too (torch.empty otherwise).
    Work goes on `stream` (default: torch's current stream of V's device, which is made current for the call)."""
    import torch as t
    lib = load_library()

    def vec(x, n, what):
        if not (isinstance(x, t.Tensor) and x.is_cuda and x.dtype == t.float64 and x.is_contiguous()
                and x.numel() == n and x.device == V.device):
            raise TypeError(f"{what} must be a contiguous float64 CUDA tensor of {n} values on V's device")
        return x

    if not (isinstance(V, t.Tensor) and V.is_cuda and V.dtype == t.float64 and V.is_contiguous() and V.dim() == 2
            and V.shape[0] == V.shape[1]):
        raise TypeError("V must be a contiguous square float64 CUDA tensor")
    N = int(V.shape[0])
    grad = vec(grad, N, "grad")
    if (dx is None) != (dg is None):
        raise ValueError("dx and dg must both be given or both be None")
    if dx is not None:
        dx, dg = vec(dx, N, "dx"), vec(dg, N, "dg")
    direction = t.empty(N, dtype=t.float64, device=V.device) if direction is None else vec(direction, N, "direction")
    edm = t.empty(2, dtype=t.float64, device=V.device) if edm is None else vec(edm, 2, "edm")
    err = C.create_string_buffer(512)
    with t.cuda.device(V.device):
        if stream is None:
            stream = t.cuda.current_stream(V.device).cuda_stream
        st = lib.phylino_variable_metric_step_static(
            C.c_void_p(stream), N, V.data_ptr(), dx.data_ptr() if dx is not None else None,
            dg.data_ptr() if dg is not None else None, grad.data_ptr(), direction.data_ptr(), edm.data_ptr(),
            err, len(err))
    if st != 0:
        raise PhylinoError(st, err.value.decode())
    return direction, edm


class Phylino:
    """One fit context (phylino_ctx).  Method names follow the C entry points.

    `model` / `events` are `workloads.ModelSpec` / `workloads.DatasetEvents`-shaped objects (plain
    attribute containers); device-side arguments are float64 CUDA tensors.
    """

    def __init__(self, device: int = 0, stream: Optional[int] = None):
        import torch
        self._torch = torch
        self._lib = load_library()
        if not torch.cuda.is_available():
            raise PhylinoError(5, "no CUDA device: this path has no CPU fallback")
        self.device = int(device)
        if stream is None:
            stream = torch.cuda.current_stream(self.device).cuda_stream
        self._ctx = C.c_void_p()
        st = self._lib.phylino_create(self.device, C.c_void_p(stream), C.byref(self._ctx))
        if st != 0:
            raise PhylinoError(st, "phylino_create failed")
        self.n_params = 0

    # -- plumbing ------------------------------------------------------------------------------
    def _check(self, st: int):
        if st != 0:
            raise PhylinoError(st, self._lib.phylino_last_error(self._ctx).decode())

    def close(self):
        if getattr(self, "_ctx", None) is not None and self._ctx:
            self._lib.phylino_destroy(self._ctx)
            self._ctx = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def __enter__(self):
        return self

    def __exit__(self, *exc):
        self.close()

    def _dev_params(self, params):
        t = self._torch
        if not (isinstance(params, t.Tensor) and params.is_cuda and params.dtype == t.float64
                and params.is_contiguous() and params.device.index == self.device):
            raise TypeError("params must be a contiguous float64 CUDA tensor on the context's device")
        if params.dim() != 2 or params.shape[1] != self.param_width:
            raise ValueError(f"params must be [P, {self.param_width}], got {tuple(params.shape)}")
        return params

    # -- phylino_set_model ---------------------------------------------------------------------
    def set_model(self, model):
        keep = []

        def arr(a, dt):
            a = np.ascontiguousarray(a, dtype=dt)
            keep.append(a)
            return a.ctypes.data

        n_ds = len(model.datasets)
        ds_arr = (_Dataset * n_ds)()
        for d, ds in enumerate(model.datasets):
            bk_arr = (_Bkg * max(1, len(ds.bkg)))()
            for k, bk in enumerate(ds.bkg):
                bk_arr[k].idx_rate = int(bk.idx_rate)
                bk_arr[k].tmpl = arr(bk.tmpl, np.float64)
                bk_arr[k].idx_shape = None if bk.idx_shape is None else arr(bk.idx_shape, np.int32)
            keep.append(bk_arr)
            ds_arr[d].n_bins = int(ds.n_bins)
            ds_arr[d].idx_a = (C.c_int32 * 3)(*[int(i) for i in ds.idx_a])
            ds_arr[d].idx_signorm = int(ds.idx_signorm)
            ds_arr[d].norm = float(ds.norm)
            ds_arr[d].idx_flux = None if ds.idx_flux is None else arr(ds.idx_flux, np.int32)
            ds_arr[d].n_bkg = len(ds.bkg)
            ds_arr[d].bkg = C.cast(bk_arr, C.POINTER(_Bkg))
        m = _Model()
        m.osc_model = int(model.osc_model)
        m.ordering = int(model.ordering)
        m.n_params = int(model.n_params)
        m.n_datasets = n_ds
        m.idx_osc = (C.c_int32 * 6)(*[int(i) for i in model.idx_osc])
        m.fixed_osc = (C.c_double * 6)(*[float(x) for x in model.fixed_osc])
        m.datasets = C.cast(ds_arr, C.POINTER(_Dataset))
        m.prior_mean = None if model.prior_mean is None else arr(model.prior_mean, np.float64)
        m.prior_sigma = None if model.prior_sigma is None else arr(model.prior_sigma, np.float64)
        self._check(self._lib.phylino_set_model(self._ctx, C.byref(m)))
        self.n_params = int(model.n_params)
        self._sizes = None
        del keep

    # -- phylino_load_events -------------------------------------------------------------------
    def load_events(self, dataset: int, e_nu, e_vis, weight, core, baseline_m, edges):
        e_nu = np.ascontiguousarray(e_nu, dtype=np.float32)
        e_vis = np.ascontiguousarray(e_vis, dtype=np.float32)
        w = None if weight is None else np.ascontiguousarray(weight, dtype=np.float32)
        c = None if core is None else np.ascontiguousarray(core, dtype=np.int32)
        L = np.ascontiguousarray(baseline_m, dtype=np.float64)
        ed = np.ascontiguousarray(edges, dtype=np.float64)
        if e_vis.shape != e_nu.shape or (w is not None and w.shape != e_nu.shape) \
                or (c is not None and c.shape != e_nu.shape):
            raise ValueError("event arrays must have the same length")
        self._check(self._lib.phylino_load_events(
            self._ctx, int(dataset), int(e_nu.shape[0]), _np_ptr(e_nu), _np_ptr(e_vis), _np_ptr(w),
            _np_ptr(c), int(L.shape[0]), _np_ptr(L), int(ed.shape[0] - 1), _np_ptr(ed)))

    def load_workload(self, wl):
        """set_model + load_events for every dataset of a `workloads.Workload`."""
        self.set_model(wl.model)
        functions = list(getattr(wl.model, "functions", None) or [])
        if functions:
            self.set_functions(functions)
        blocks = list(getattr(wl.model, "prior_blocks", None) or [])
        if blocks:
            self.set_prior_blocks(blocks)
        for d, ds in enumerate(wl.model.datasets):
            fm = getattr(ds, "flux_model", None)
            if fm is not None:
                self.set_flux_model(d, fm.idx_par, fm.lo, fm.width)
        if int(getattr(wl.model, "energy_correction", 0)):
            self.set_energy_correction_mode(1)
        for d, e in enumerate(wl.events):
            self.load_events(d, e.e_nu, e.e_vis, e.w, e.core, e.L_m, e.edges)

    # -- sizes ---------------------------------------------------------------------------------
    def _size_cache(self):
        # (total_bins, param_width): fixed between set_model / set_transform calls; asked once, because a
        # single-point host call is short enough for two extra library calls to show
        if getattr(self, "_sizes", None) is None:
            self._sizes = (int(self._lib.phylino_total_bins(self._ctx)), int(self._lib.phylino_param_width(self._ctx)))
        return self._sizes

    @property
    def total_bins(self) -> int:
        return self._size_cache()[0]

    @property
    def total_events(self) -> int:
        return int(self._lib.phylino_total_events(self._ctx))

    @property
    def launch_count(self) -> int:
        return int(self._lib.phylino_launch_count(self._ctx))

    def set_tuning(self, unit_events: int = 0, chunk_groups: int = 0, max_warps: int = 0):
        self._check(self._lib.phylino_set_tuning(self._ctx, int(unit_events), int(chunk_groups), int(max_warps)))

    def set_energy_correction_mode(self, mode: int):
        """0: per event before binning (default); 1: on the binned spectrum (PAPER.md:177 step 3)."""
        self._check(self._lib.phylino_set_energy_correction_mode(self._ctx, int(mode)))

    def set_flux_model(self, dataset: int, idx_par, lo: float = 1.0, width: float = 0.25):
        """fine-grid flux parameters of one dataset; idx_par empty removes the model."""
        idx = np.ascontiguousarray(idx_par, dtype=np.int32)
        self._check(self._lib.phylino_set_flux_model(self._ctx, int(dataset), int(idx.size),
                                                     idx.ctypes.data if idx.size else None, float(lo), float(width)))

    def set_schedule(self, mode: int = 0):
        """0 library's choice, 1 always setup/spectra/finalize kernels, 2 single launch for <= 16 points."""
        self._check(self._lib.phylino_set_schedule(self._ctx, int(mode)))

    def reserve(self, max_points: int):
        self._check(self._lib.phylino_reserve(self._ctx, int(max_points)))

    # -- phylino_spectra / phylino_nll / phylino_event_bins (device buffers, asynchronous) -------
    def spectra(self, params, out=None):
        t = self._torch
        p = self._dev_params(params)
        if out is None:
            out = t.empty((p.shape[0], self.total_bins), dtype=t.float64, device=p.device)
        assert out.is_cuda and out.dtype == t.float64 and out.is_contiguous() \
            and out.numel() == p.shape[0] * self.total_bins
        self._check(self._lib.phylino_spectra(self._ctx, int(p.shape[0]), p.data_ptr(), out.data_ptr()))
        return out

    def nll(self, params, data, out=None):
        t = self._torch
        p = self._dev_params(params)
        if not (isinstance(data, t.Tensor) and data.is_cuda and data.dtype == t.float64
                and data.is_contiguous() and data.numel() == self.total_bins):
            raise TypeError(f"data must be a contiguous float64 CUDA tensor of {self.total_bins} counts")
        if out is None:
            out = t.empty((p.shape[0],), dtype=t.float64, device=p.device)
        assert out.is_cuda and out.dtype == t.float64 and out.is_contiguous() and out.numel() == p.shape[0]
        self._check(self._lib.phylino_nll(self._ctx, int(p.shape[0]), p.data_ptr(), data.data_ptr(),
                                          out.data_ptr()))
        return out

    def nll_ensemble(self, params, data, out=None):
        """data: float64 CUDA tensor [E, total_bins] -> nll [P, E]."""
        t = self._torch
        p = self._dev_params(params)
        if not (isinstance(data, t.Tensor) and data.is_cuda and data.dtype == t.float64 and data.is_contiguous()
                and data.dim() == 2 and data.shape[1] == self.total_bins):
            raise TypeError(f"data must be a contiguous float64 CUDA tensor [E, {self.total_bins}]")
        E = int(data.shape[0])
        if out is None:
            out = t.empty((p.shape[0], E), dtype=t.float64, device=p.device)
        assert out.is_cuda and out.dtype == t.float64 and out.is_contiguous() and out.numel() == p.shape[0] * E
        self._check(self._lib.phylino_nll_ensemble(self._ctx, int(p.shape[0]), p.data_ptr(), E, data.data_ptr(),
                                                   out.data_ptr()))
        return out

    def _dev_vec(self, x, n, what):
        t = self._torch
        if not (isinstance(x, t.Tensor) and x.is_cuda and x.dtype == t.float64 and x.is_contiguous() and x.numel() == n):
            raise TypeError(f"{what} must be a contiguous float64 CUDA tensor of {n} values")
        return x

    def draw_pseudo_data(self, mu, n_experiments: int, seed: int, out=None):
        """mu: float64 CUDA tensor [total_bins] -> Poisson counts [E, total_bins] (float64)."""
        t = self._torch
        mu = self._dev_vec(mu, self.total_bins, "mu")
        E = int(n_experiments)
        if out is None:
            out = t.empty((E, self.total_bins), dtype=t.float64, device=mu.device)
        assert out.is_cuda and out.dtype == t.float64 and out.is_contiguous() and out.numel() == E * self.total_bins
        self._check(self._lib.phylino_draw_pseudo_data(self._ctx, mu.data_ptr(), E, int(seed) & (2 ** 64 - 1), out.data_ptr()))
        return out

    def ordering_scan(self, scan_param: int, grid, theta, data, out=None):
        """grid [n_grid], theta [param_width], data [total_bins] (float64 CUDA) -> nll [2, n_grid]: normal, inverted."""
        t = self._torch
        n = int(grid.numel())
        grid = self._dev_vec(grid, n, "grid")
        theta = self._dev_vec(theta, self.param_width, "theta")
        data = self._dev_vec(data, self.total_bins, "data")
        if out is None:
            out = t.empty((2, n), dtype=t.float64, device=grid.device)
        assert out.is_cuda and out.dtype == t.float64 and out.is_contiguous() and out.numel() == 2 * n
        self._check(self._lib.phylino_ordering_scan(self._ctx, n, int(scan_param), grid.data_ptr(), theta.data_ptr(),
                                                    data.data_ptr(), out.data_ptr()))
        return out

    def nll_gradient(self, theta, step, data, nll0=None, grad=None):
        """theta, step [param_width], data [total_bins] (float64 CUDA) -> (nll(theta) [1], grad [param_width])."""
        t = self._torch
        N = self.param_width
        theta, step = self._dev_vec(theta, N, "theta"), self._dev_vec(step, N, "step")
        data = self._dev_vec(data, self.total_bins, "data")
        if nll0 is None:
            nll0 = t.empty(1, dtype=t.float64, device=theta.device)
        if grad is None:
            grad = t.empty(N, dtype=t.float64, device=theta.device)
        nll0, grad = self._dev_vec(nll0, 1, "nll0"), self._dev_vec(grad, N, "grad")
        self._check(self._lib.phylino_nll_gradient(self._ctx, theta.data_ptr(), step.data_ptr(), data.data_ptr(),
                                                   nll0.data_ptr(), grad.data_ptr()))
        return nll0, grad

    def variable_metric_step(self, V, grad, dx=None, dg=None):
        """One variable-metric step: V [N, N] float64 CUDA, updated IN PLACE from the last move dx and
        gradient change dg (both or neither); returns (direction [N], edm [2] = (edm, update skipped))."""
        t = self._torch
        if not (isinstance(V, t.Tensor) and V.is_cuda and V.dtype == t.float64 and V.is_contiguous() and V.dim() == 2
                and V.shape[0] == V.shape[1]):
            raise TypeError("V must be a contiguous square float64 CUDA tensor")
        N = int(V.shape[0])
        grad = self._dev_vec(grad, N, "grad")
        if (dx is None) != (dg is None):
            raise ValueError("dx and dg must both be given or both be None")
        if dx is not None:
            dx, dg = self._dev_vec(dx, N, "dx"), self._dev_vec(dg, N, "dg")
        direction = t.empty(N, dtype=t.float64, device=V.device)
        edm = t.empty(2, dtype=t.float64, device=V.device)
        self._check(self._lib.phylino_variable_metric_step(
            self._ctx, N, V.data_ptr(), dx.data_ptr() if dx is not None else None,
            dg.data_ptr() if dg is not None else None, grad.data_ptr(), direction.data_ptr(), edm.data_ptr()))
        return direction, edm

    def expectation(self, params, out=None):
        t = self._torch
        p = self._dev_params(params)
        if out is None:
            out = t.empty((p.shape[0], self.total_bins), dtype=t.float64, device=p.device)
        assert out.is_cuda and out.dtype == t.float64 and out.is_contiguous() \
            and out.numel() == p.shape[0] * self.total_bins
        self._check(self._lib.phylino_expectation(self._ctx, int(p.shape[0]), p.data_ptr(), out.data_ptr()))
        return out

    def set_functions(self, functions: Sequence = ()):
        """constrained functions of theta: each has .offset and .terms = [(coef, idx, power), ...];
        a prior block names function f as n_params + f.  Empty clears."""
        functions = list(functions)
        keep = []
        arr = (_Function * max(1, len(functions)))()
        for k, f in enumerate(functions):
            ta = (_Monomial * max(1, len(f.terms)))()
            for j, (coef, idx, power) in enumerate(f.terms):
                idx = np.ascontiguousarray(idx, dtype=np.int32)
                power = np.ascontiguousarray(power, dtype=np.int32)
                if idx.shape != power.shape or idx.ndim != 1:
                    raise ValueError("function term: idx and power must be 1-d arrays of equal length")
                keep += [idx, power]
                ta[j].coef = float(coef)
                ta[j].n_factors = int(idx.shape[0])
                ta[j].idx = idx.ctypes.data
                ta[j].power = power.ctypes.data
            keep.append(ta)
            arr[k].offset = float(f.offset)
            arr[k].n_terms = len(f.terms)
            arr[k].terms = C.cast(ta, C.POINTER(_Monomial))
        self._check(self._lib.phylino_set_functions(self._ctx, len(functions), arr if functions else None))

    def set_prior_blocks(self, blocks: Sequence = ()):
        """blocks: objects with .idx [n], .mean [n], .inv_cov [n, n] (workloads.PriorBlock)."""
        keep = []
        arr = (_PriorBlock * max(1, len(blocks)))()
        for k, b in enumerate(blocks):
            i = np.ascontiguousarray(b.idx, dtype=np.int32)
            m = np.ascontiguousarray(b.mean, dtype=np.float64)
            v = np.ascontiguousarray(b.inv_cov, dtype=np.float64)
            if m.shape != i.shape or v.shape != (i.size, i.size):
                raise ValueError("prior block: idx [n], mean [n], inv_cov [n, n]")
            keep += [i, m, v]
            arr[k].n, arr[k].idx, arr[k].mean, arr[k].inv_cov = int(i.size), i.ctypes.data, m.ctypes.data, v.ctypes.data
        self._check(self._lib.phylino_set_prior_blocks(self._ctx, len(blocks), arr if blocks else None))

    def set_transform(self, spec=None):
        """spec: workloads.TransformSpec (n_u, copy_src, copy_const, blocks) or None to remove the layer."""
        self._sizes = None
        if spec is None:
            self._check(self._lib.phylino_set_transform(self._ctx, 0, None, None, 0, None))
            return
        keep = []

        def arr(a, dt):
            a = np.ascontiguousarray(a, dtype=dt)
            keep.append(a)
            return a.ctypes.data
        blocks = list(spec.blocks)
        tb = (_TransformBlock * max(1, len(blocks)))()
        for k, b in enumerate(blocks):
            tb[k].n_out, tb[k].n_in = len(b.idx_out), len(b.idx_in)
            if np.shape(b.matrix) != (tb[k].n_out, tb[k].n_in):
                raise ValueError("transform block: matrix must be [n_out, n_in]")
            tb[k].idx_out, tb[k].idx_in = arr(b.idx_out, np.int32), arr(b.idx_in, np.int32)
            tb[k].offset, tb[k].centre = arr(b.offset, np.float64), arr(b.centre, np.float64)
            tb[k].matrix = arr(b.matrix, np.float64)
        self._check(self._lib.phylino_set_transform(self._ctx, int(spec.n_u), arr(spec.copy_src, np.int32),
                                                    arr(spec.copy_const, np.float64), len(blocks),
                                                    tb if blocks else None))

    @property
    def param_width(self) -> int:
        return self._size_cache()[1]

    def set_caching(self, on: bool = True):
        self._check(self._lib.phylino_set_caching(self._ctx, int(bool(on))))

    def last_plan(self):
        """(virtual points, energy-scale classes) of the last host call that used the cache; (0, 0) if dense."""
        v, c = C.c_int64(0), C.c_int64(0)
        self._check(self._lib.phylino_last_plan(self._ctx, C.byref(v), C.byref(c)))
        return int(v.value), int(c.value)

    def last_medium_phase(self) -> float:
        """fraction of the last call's event x point evaluations whose first term took the no-reduction form"""
        v = C.c_double(0.0)
        self._check(self._lib.phylino_last_medium_phase(self._ctx, C.byref(v)))
        return float(v.value)

    def last_small_phase(self) -> float:
        """fraction of the last call's event x point evaluations whose last term took the small-phase form"""
        v = C.c_double(0.0)
        self._check(self._lib.phylino_last_small_phase(self._ctx, C.byref(v)))
        return float(v.value)

    def set_timing(self, on: bool = True):
        self._check(self._lib.phylino_set_timing(self._ctx, int(bool(on))))

    def last_kernel_ms(self):
        """(setup, spectra, finalize) kernel ms of the last call; waits for it to finish."""
        ms = (C.c_float * 3)()
        self._check(self._lib.phylino_last_kernel_ms(self._ctx, ms))
        return float(ms[0]), float(ms[1]), float(ms[2])

    def event_bins(self, params):
        t = self._torch
        p = self._dev_params(params)
        out = t.empty((p.shape[0], self.total_events), dtype=t.int32, device=p.device)
        self._check(self._lib.phylino_event_bins(self._ctx, int(p.shape[0]), p.data_ptr(), out.data_ptr()))
        return out

    # -- host-buffer entry points (synchronous, copies inside) ---------------------------------
    def nll_host(self, params: np.ndarray, data: np.ndarray, out: Optional[np.ndarray] = None) -> np.ndarray:
        p = np.ascontiguousarray(params, dtype=np.float64)
        d = np.ascontiguousarray(data, dtype=np.float64)
        if p.ndim != 2 or p.shape[1] != self.param_width or d.shape != (self.total_bins,):
            raise ValueError("bad shapes")
        if out is None:
            out = np.empty(p.shape[0], dtype=np.float64)
        self._check(self._lib.phylino_nll_host(self._ctx, int(p.shape[0]), p.ctypes.data, d.ctypes.data,
                                               out.ctypes.data))
        return out

    def spectra_host(self, params: np.ndarray, out: Optional[np.ndarray] = None) -> np.ndarray:
        p = np.ascontiguousarray(params, dtype=np.float64)
        if p.ndim != 2 or p.shape[1] != self.param_width:
            raise ValueError("bad shapes")
        if out is None:
            out = np.empty((p.shape[0], self.total_bins), dtype=np.float64)
        self._check(self._lib.phylino_spectra_host(self._ctx, int(p.shape[0]), p.ctypes.data, out.ctypes.data))
        return out

    def launch_floor(self, reps: int = 200) -> float:
        """microseconds per (empty-kernel launch + stream synchronise) on this context's stream."""
        v = C.c_double(0.0)
        self._check(self._lib.phylino_launch_floor(self._ctx, int(reps), C.byref(v)))
        return float(v.value)

    def hbm_read_floor(self, nbytes: int, reps: int = 10) -> float:
        """microseconds of one kernel that only reads nbytes from HBM (L2 flushed), best of reps"""
        v = C.c_double(0.0)
        self._check(self._lib.phylino_hbm_read_floor(self._ctx, int(nbytes), int(reps), C.byref(v)))
        return float(v.value)

    def peak_fp64(self, iters: int = 4096) -> float:
        v = C.c_double(0.0)
        self._check(self._lib.phylino_peak_fp64(self._ctx, int(iters), C.byref(v)))
        return float(v.value)
