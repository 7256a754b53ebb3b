"""ctypes front-end of the CPU oracle (oracle.c).  TEST INFRASTRUCTURE ONLY.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may
import this.  It never imports paper_2502_15253_b200 and vice versa; the only module both sides
use is `workloads` (seeded inputs, no arithmetic of the method).
"""
from __future__ import annotations

import ctypes as C
import os
import subprocess
from typing import List, Sequence

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "oracle.c")
_LIB = os.path.join(_HERE, "liboracle.so")
_CFLAGS = ["-O2", "-std=c11", "-mfma", "-ffp-contract=off", "-fopenmp", "-shared", "-fPIC"]


def build(force: bool = False) -> str:
    """Compile oracle.c with gcc (building the checker is not using it)."""
    stale = (not os.path.exists(_LIB)) or any(
        os.path.getmtime(os.path.join(_HERE, f)) > os.path.getmtime(_LIB) for f in ("oracle.c", "oracle.h"))
    if force or stale:
        tmp = _LIB + f".tmp{os.getpid()}"
        subprocess.check_call(["gcc", *_CFLAGS, _SRC, "-o", tmp, "-lm"])
        os.replace(tmp, _LIB)
    return _LIB


class _Events(C.Structure):
    _fields_ = [("n", C.c_int64), ("e_nu", C.c_void_p), ("e_vis", C.c_void_p), ("w", C.c_void_p),
                ("core", C.c_void_p), ("n_cores", C.c_int32), ("L_m", C.c_void_p),
                ("n_bins", C.c_int32), ("edges", C.c_void_p)]


class _Bkg(C.Structure):
    _fields_ = [("idx_rate", C.c_int32), ("tmpl", C.c_void_p), ("idx_shape", C.c_void_p)]


class _Dataset(C.Structure):
    _fields_ = [("n_bins", C.c_int32), ("idx_a", C.c_int32 * 3), ("idx_signorm", C.c_int32),
                ("norm", C.c_double), ("idx_flux", C.c_void_p), ("n_bkg", C.c_int32),
                ("bkg", C.POINTER(_Bkg)), ("n_flux_par", C.c_int32), ("idx_flux_par", C.c_void_p),
                ("flux_lo", C.c_double), ("flux_width", C.c_double)]


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
                ("datasets", C.POINTER(_Dataset)), ("prior_mean", C.c_void_p), ("prior_sigma", C.c_void_p),
                ("n_prior_blocks", C.c_int32), ("prior_blocks", C.POINTER(_PriorBlock)),
                ("energy_correction", C.c_int32),
                ("n_functions", C.c_int32), ("functions", C.POINTER(_Function))]


_lib = None


def _load():
    global _lib
    if _lib is None:
        lib = C.CDLL(build())
        dp = C.POINTER(C.c_double)
        lib.orc_terms.restype = C.c_int
        lib.orc_terms.argtypes = [C.POINTER(_Model), dp, dp, dp]
        lib.orc_pee.restype = C.c_double
        lib.orc_pee.argtypes = [C.c_int, dp, dp, C.c_double, C.c_double]
        lib.orc_escale.restype = C.c_double
        lib.orc_escale.argtypes = [C.c_double] * 4
        lib.orc_bin.restype = C.c_int32
        lib.orc_bin.argtypes = [dp, C.c_int32, C.c_double]
        lib.orc_dev.restype = C.c_double
        lib.orc_dev.argtypes = [C.c_double, C.c_double]
        lib.orc_spectra.restype = C.c_int
        lib.orc_spectra.argtypes = [C.POINTER(_Model), C.POINTER(_Events), C.c_int32, dp, dp, C.c_int]
        lib.orc_event_bins.restype = C.c_int
        lib.orc_event_bins.argtypes = [C.POINTER(_Model), C.POINTER(_Events), C.c_int32, dp,
                                       C.POINTER(C.c_int32)]
        lib.orc_expectation.restype = C.c_int
        lib.orc_expectation.argtypes = [C.POINTER(_Model), C.POINTER(dp), C.c_int32, dp, dp, dp]
        lib.orc_correct_spectra.restype = C.c_int
        lib.orc_correct_spectra.argtypes = [C.POINTER(_Model), C.POINTER(dp), C.c_int32, dp, dp, dp]
        lib.orc_escale_inverse.restype = C.c_double
        lib.orc_escale_inverse.argtypes = [C.c_double] * 4
        lib.orc_rebin_quadratic.restype = C.c_int
        lib.orc_rebin_quadratic.argtypes = [C.c_int32, dp, dp, C.c_int32, dp, dp]
        lib.orc_flux_scales.restype = C.c_int
        lib.orc_flux_scales.argtypes = [C.POINTER(_Dataset), dp, dp, dp]
        lib.orc_nll_from_mu.restype = C.c_int
        lib.orc_nll_from_mu.argtypes = [C.POINTER(_Model), C.c_int32, dp, dp, dp, dp]
        lib.orc_variable_metric_step.restype = C.c_int
        lib.orc_variable_metric_step.argtypes = [C.c_int32, dp, dp, dp, dp, dp, dp]
        lib.orc_function_value.restype = C.c_double
        lib.orc_function_value.argtypes = [C.POINTER(_Function), dp]
        lib.orc_nll.restype = C.c_int
        lib.orc_nll.argtypes = [C.POINTER(_Model), C.POINTER(_Events), C.c_int32, dp, dp, dp, C.c_int]
        lib.orc_transform.restype = C.c_int
        lib.orc_transform.argtypes = [C.c_int32, C.c_int32, C.c_void_p, C.c_void_p, C.c_int32,
                                      C.POINTER(_TransformBlock), C.c_int32, dp, dp]
        lib.orc_philox4x32_10.restype = None
        lib.orc_philox4x32_10.argtypes = [C.POINTER(C.c_uint32), C.POINTER(C.c_uint32), C.POINTER(C.c_uint32)]
        lib.orc_uniform53.restype = C.c_double
        lib.orc_uniform53.argtypes = [C.c_uint64, C.c_uint32, C.c_uint32]
        lib.orc_poisson_norm.restype = C.c_double
        lib.orc_poisson_norm.argtypes = [C.c_double]
        lib.orc_poisson_inv.restype = C.c_double
        lib.orc_poisson_inv.argtypes = [C.c_double, C.c_double, C.c_double]
        lib.orc_draw_pseudo_data.restype = C.c_int
        lib.orc_draw_pseudo_data.argtypes = [C.c_int64, dp, C.c_int32, C.c_uint64, dp]
        lib.orc_max_threads.restype = C.c_int
        _lib = lib
    return _lib


def _dp(a: np.ndarray):
    return a.ctypes.data_as(C.POINTER(C.c_double))


def _f64(a) -> np.ndarray:
    return np.ascontiguousarray(a, dtype=np.float64)


class Oracle:
    """Binds one `workloads.ModelSpec` (+ optionally its event lists) to the C oracle."""

    def __init__(self, model, events: Sequence = ()):
        self._keep: List[object] = []          # numpy arrays the C structs point into
        self.model = model
        self._m = self._marshal_model(model)
        self._ev = self._marshal_events(events) if len(events) else None
        self.n_params = model.n_params
        self.total_bins = sum(d.n_bins for d in model.datasets)
        self.n_events = sum(e.n for e in events)
        self.bin_level = int(getattr(model, "energy_correction", 0)) == 1
        # bin edges per dataset (the bin-level steps need them): from the events if given
        self._edges = None
        if len(events):
            arrs = [np.ascontiguousarray(e.edges, dtype=np.float64) for e in events]
            self._keep.extend(arrs)
            self._edges = (C.POINTER(C.c_double) * len(arrs))(*[_dp(a) for a in arrs])

    # -- marshalling ---------------------------------------------------------------------------
    def _arr(self, a, dtype):
        a = np.ascontiguousarray(a, dtype=dtype)
        self._keep.append(a)
        return a.ctypes.data

    def _marshal_model(self, model) -> _Model:
        ds_arr = (_Dataset * len(model.datasets))()
        for d, ds in enumerate(model.datasets):
            bk_arr = (_Bkg * max(1, len(ds.bkg)))()
            for k, bk in enumerate(ds.bkg):
                bk_arr[k].idx_rate = int(bk.idx_rate)
                bk_arr[k].tmpl = self._arr(bk.tmpl, np.float64)
                bk_arr[k].idx_shape = None if bk.idx_shape is None else self._arr(bk.idx_shape, np.int32)
            self._keep.append(bk_arr)
            ds_arr[d].n_bins = int(ds.n_bins)
            ds_arr[d].idx_a = (C.c_int32 * 3)(*[int(i) for i in ds.idx_a])
            ds_arr[d].idx_signorm = int(ds.idx_signorm)
            ds_arr[d].norm = float(ds.norm)
            ds_arr[d].idx_flux = None if ds.idx_flux is None else self._arr(ds.idx_flux, np.int32)
            ds_arr[d].n_bkg = len(ds.bkg)
            ds_arr[d].bkg = C.cast(bk_arr, C.POINTER(_Bkg))
            fm = getattr(ds, "flux_model", None)
            if fm is not None:
                ds_arr[d].n_flux_par = len(fm.idx_par)
                ds_arr[d].idx_flux_par = self._arr(fm.idx_par, np.int32)
                ds_arr[d].flux_lo, ds_arr[d].flux_width = float(fm.lo), float(fm.width)
        self._keep.append(ds_arr)
        self._ds_arr = ds_arr
        m = _Model()
        m.osc_model = int(model.osc_model)
        m.ordering = int(model.ordering)
        m.n_params = int(model.n_params)
        m.n_datasets = len(model.datasets)
        m.idx_osc = (C.c_int32 * 6)(*[int(i) for i in model.idx_osc])
        m.fixed_osc = (C.c_double * 6)(*[float(x) for x in model.fixed_osc])
        m.datasets = C.cast(ds_arr, C.POINTER(_Dataset))
        m.prior_mean = None if model.prior_mean is None else self._arr(model.prior_mean, np.float64)
        m.prior_sigma = None if model.prior_sigma is None else self._arr(model.prior_sigma, np.float64)
        blocks = list(getattr(model, "prior_blocks", None) or [])
        pb = (_PriorBlock * max(1, len(blocks)))()
        for k, b in enumerate(blocks):
            n = len(b.idx)
            assert np.shape(b.mean) == (n,) and np.shape(b.inv_cov) == (n, n)
            pb[k].n = n
            pb[k].idx = self._arr(b.idx, np.int32)
            pb[k].mean = self._arr(b.mean, np.float64)
            pb[k].inv_cov = self._arr(b.inv_cov, np.float64)
        self._keep.append(pb)
        m.n_prior_blocks = len(blocks)
        m.prior_blocks = C.cast(pb, C.POINTER(_PriorBlock)) if blocks else None
        m.energy_correction = int(getattr(model, "energy_correction", 0))
        funcs = list(getattr(model, "functions", None) or [])
        fa = (_Function * max(1, len(funcs)))()
        for k, f in enumerate(funcs):
            ta = (_Monomial * max(1, len(f.terms)))()
            for j, (coef, idx, power) in enumerate(f.terms):
                assert len(idx) == len(power)
                ta[j].coef = float(coef)
                ta[j].n_factors = len(idx)
                ta[j].idx = self._arr(idx, np.int32)
                ta[j].power = self._arr(power, np.int32)
            self._keep.append(ta)
            fa[k].offset = float(f.offset)
            fa[k].n_terms = len(f.terms)
            fa[k].terms = C.cast(ta, C.POINTER(_Monomial))
        self._keep.append(fa)
        m.n_functions = len(funcs)
        m.functions = C.cast(fa, C.POINTER(_Function)) if funcs else None
        return m

    def _marshal_events(self, events):
        arr = (_Events * len(events))()
        for d, e in enumerate(events):
            arr[d].n = e.n
            arr[d].e_nu = self._arr(e.e_nu, np.float32)
            arr[d].e_vis = self._arr(e.e_vis, np.float32)
            arr[d].w = None if e.w is None else self._arr(e.w, np.float32)
            arr[d].core = None if e.core is None else self._arr(e.core, np.int32)
            arr[d].n_cores = len(e.L_m)
            arr[d].L_m = self._arr(e.L_m, np.float64)
            arr[d].n_bins = e.n_bins
            arr[d].edges = self._arr(e.edges, np.float64)
        return arr

    def _params(self, params):
        p = _f64(params)
        if p.ndim == 1:
            p = p[None, :]
        assert p.shape[1] == self.n_params, (p.shape, self.n_params)
        return p

    # -- O1/O2 ---------------------------------------------------------------------------------
    def terms(self, theta):
        th = _f64(theta)
        A = np.zeros(3)
        m = np.zeros(3)
        S = _load().orc_terms(C.byref(self._m), _dp(th), _dp(A), _dp(m))
        assert S > 0
        return A[:S].copy(), m[:S].copy()

    # -- O3 ------------------------------------------------------------------------------------
    def spectra_raw(self, params, n_threads: int = 0) -> np.ndarray:
        """step 1 of PAPER.md:177; with energy_correction = 1 binned under the identity energy scale"""
        p = self._params(params)
        hist = np.zeros((p.shape[0], self.total_bins))
        rc = _load().orc_spectra(C.byref(self._m), self._ev, p.shape[0], _dp(p), _dp(hist), n_threads)
        assert rc == 0, rc
        return hist

    def spectra(self, params, n_threads: int = 0) -> np.ndarray:
        """the signal spectrum the product's spectra call returns: step 1, plus the bin-level energy correction
        (step 3, no flux re-scaling) when energy_correction = 1"""
        hist = self.spectra_raw(params, n_threads)
        if not self.bin_level:
            return hist
        p = self._params(params)
        out = np.zeros_like(hist)
        rc = _load().orc_correct_spectra(C.byref(self._m), self._edges, p.shape[0], _dp(p), _dp(hist), _dp(out))
        assert rc == 0, rc
        return out

    def event_bins(self, params) -> np.ndarray:
        p = self._params(params)
        bins = np.zeros((p.shape[0], self.n_events), dtype=np.int32)
        rc = _load().orc_event_bins(C.byref(self._m), self._ev, p.shape[0], _dp(p),
                                    bins.ctypes.data_as(C.POINTER(C.c_int32)))
        assert rc == 0, rc
        return bins

    # -- O4 / O5 -------------------------------------------------------------------------------
    def expectation(self, params, hist) -> np.ndarray:
        """hist: the step-1 spectra (with energy_correction = 1: spectra_raw, not spectra)"""
        p = self._params(params)
        h = _f64(hist).reshape(p.shape[0], self.total_bins)
        mu = np.zeros_like(h)
        rc = _load().orc_expectation(C.byref(self._m), self._edges, p.shape[0], _dp(p), _dp(h), _dp(mu))
        assert rc == 0, rc
        return mu

    def flux_scales(self, dataset: int, theta) -> np.ndarray:
        th = _f64(theta)
        f = np.zeros(self.model.datasets[dataset].n_bins)
        ed = np.ascontiguousarray(self._keep_edges(dataset))
        rc = _load().orc_flux_scales(C.byref(self._ds_arr[dataset]), _dp(ed), _dp(th), _dp(f))
        assert rc == 0, rc
        return f

    def _keep_edges(self, dataset: int) -> np.ndarray:
        n = self.model.datasets[dataset].n_bins
        return np.ctypeslib.as_array(self._edges[dataset], shape=(n + 1,)).copy()

    def function_values(self, theta) -> np.ndarray:
        """b_f(theta) of the model's constrained functions (R29) at one point."""
        th = _f64(theta)
        assert th.shape == (self.model.n_params,)
        return np.array([_load().orc_function_value(C.byref(self._m.functions[f]), _dp(th))
                         for f in range(self._m.n_functions)])

    def nll_from_mu(self, params, mu, data) -> np.ndarray:
        p = self._params(params)
        mu = _f64(mu).reshape(p.shape[0], self.total_bins)
        data = _f64(data)
        assert data.shape == (self.total_bins,)
        out = np.zeros(p.shape[0])
        rc = _load().orc_nll_from_mu(C.byref(self._m), p.shape[0], _dp(p), _dp(mu), _dp(data), _dp(out))
        assert rc == 0, rc
        return out

    def nll(self, params, data, n_threads: int = 0) -> np.ndarray:
        p = self._params(params)
        data = _f64(data)
        assert data.shape == (self.total_bins,)
        out = np.zeros(p.shape[0])
        rc = _load().orc_nll(C.byref(self._m), self._ev, p.shape[0], _dp(p), _dp(data), _dp(out), n_threads)
        assert rc == 0, rc
        return out


# -- scalar helpers (pins) ----------------------------------------------------------------------
def pee(A, dm2, L_m: float, E_MeV: float) -> float:
    A = _f64(A)
    dm2 = _f64(dm2)
    return float(_load().orc_pee(len(A), _dp(A), _dp(dm2), float(L_m), float(E_MeV)))


def escale(a0: float, a1: float, a2: float, v: float) -> float:
    return float(_load().orc_escale(a0, a1, a2, v))


def bin_index(edges, e: float) -> int:
    ed = _f64(edges)
    return int(_load().orc_bin(_dp(ed), len(ed) - 1, float(e)))


def dev(n: float, mu: float) -> float:
    return float(_load().orc_dev(float(n), float(mu)))


def transform(spec, n_params: int, u) -> np.ndarray:
    """theta [P, n_params] from the minimiser's parameters u [P, n_u] through a workloads.TransformSpec
    (PAPER.md:171, :141)."""
    lib = _load()
    u = np.ascontiguousarray(np.atleast_2d(u), dtype=np.float64)
    assert u.shape[1] == spec.n_u
    keep = []

    def arr(a, dt):
        a = np.ascontiguousarray(a, dtype=dt)
        keep.append(a)
        return a.ctypes.data
    src = np.ascontiguousarray(spec.copy_src, dtype=np.int32)
    cst = np.ascontiguousarray(spec.copy_const, dtype=np.float64)
    assert src.shape == (n_params,) and cst.shape == (n_params,)
    blocks = list(spec.blocks)
    tb = (_TransformBlock * max(1, len(blocks)))()
    for k, b in enumerate(blocks):
        n_out, n_in = len(b.idx_out), len(b.idx_in)
        assert np.shape(b.matrix) == (n_out, n_in) and np.shape(b.offset) == (n_out,) and np.shape(b.centre) == (n_in,)
        tb[k].n_out, tb[k].n_in = n_out, n_in
        tb[k].idx_out, tb[k].idx_in = arr(b.idx_out, np.int32), arr(b.idx_in, np.int32)
        tb[k].offset, tb[k].centre, tb[k].matrix = arr(b.offset, np.float64), arr(b.centre, np.float64), arr(b.matrix, np.float64)
    theta = np.empty((u.shape[0], n_params), dtype=np.float64)
    rc = lib.orc_transform(n_params, spec.n_u, src.ctypes.data, cst.ctypes.data, len(blocks), tb, u.shape[0],
                           _dp(u), _dp(theta))
    if rc != 0:
        raise ValueError(f"orc_transform failed ({rc})")
    return theta


def variable_metric_step(V, grad, dx=None, dg=None):
    """One variable-metric step (R30): returns (V_new, direction, edm, skipped)."""
    V = np.array(V, dtype=np.float64, order="C", copy=True)
    N = V.shape[0]
    assert V.shape == (N, N)
    g = _f64(grad)
    d = np.zeros(N)
    edm = np.zeros(1)
    has = dx is not None and dg is not None
    a_dx, a_dg = (_f64(dx), _f64(dg)) if has else (None, None)
    rc = _load().orc_variable_metric_step(N, _dp(V), _dp(a_dx) if has else None, _dp(a_dg) if has else None, _dp(g),
                                          _dp(d), _dp(edm))
    assert rc in (0, 1), rc
    return V, d, float(edm[0]), bool(rc)


def max_threads() -> int:
    return int(_load().orc_max_threads())


# -- pseudo-experiments (R26) ---------------------------------------------
def philox4x32_10(ctr, key):
    c = (C.c_uint32 * 4)(*[int(x) for x in ctr])
    k = (C.c_uint32 * 2)(*[int(x) for x in key])
    out = (C.c_uint32 * 4)()
    _load().orc_philox4x32_10(c, k, out)
    return [int(x) for x in out]


def uniform53(seed: int, bin_index: int, experiment: int) -> float:
    return float(_load().orc_uniform53(int(seed), int(bin_index), int(experiment)))


def poisson_norm(mu: float) -> float:
    return float(_load().orc_poisson_norm(float(mu)))


def poisson_inv(mu: float, Z: float, u: float) -> float:
    return float(_load().orc_poisson_inv(float(mu), float(Z), float(u)))


def draw_pseudo_data(mu, n_experiments: int, seed: int) -> np.ndarray:
    """data [E, total_bins]: Poisson-fluctuated counts around mu [total_bins]."""
    mu = _f64(mu)
    data = np.zeros((int(n_experiments), mu.shape[0]))
    rc = _load().orc_draw_pseudo_data(mu.shape[0], _dp(mu), int(n_experiments), int(seed), _dp(data))
    assert rc == 0, rc
    return data


# -- bin-level steps (R27) ----------------------------------------------------------------
def escale_inverse(a0: float, a1: float, a2: float, t: float) -> float:
    return float(_load().orc_escale_inverse(a0, a1, a2, t))


def rebin_quadratic(src_edges, src_int, x) -> np.ndarray:
    e, h, x = _f64(src_edges), _f64(src_int), _f64(x)
    assert e.shape[0] == h.shape[0] + 1
    out = np.zeros(x.shape[0] - 1)
    rc = _load().orc_rebin_quadratic(h.shape[0], _dp(e), _dp(h), out.shape[0], _dp(x), _dp(out))
    assert rc == 0, rc
    return out

