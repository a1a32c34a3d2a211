"""Thin ctypes binding of the C-ABI in include/nmpc.h (argument marshalling only; every step runs in the CUDA library).

The function names are those of the header: nmpc_analyze, nmpc_update_params, nmpc_factor, nmpc_solve,
nmpc_ipm_solve, ...  PyTorch supplies device buffers (tensor.data_ptr()) and the CUDA stream; nothing here computes.
If libnmpc_b200.so is missing or cannot be loaded this module raises: there is no CPU fallback.
"""
from __future__ import annotations

import ctypes as C
import os

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libnmpc_b200.so")

STATUS_NAMES = ["OK", "E_ARG", "E_PATTERN", "E_ALLOC", "E_CUDA", "E_STATE", "E_NOT_SPD", "E_INERTIA", "E_MAXITER", "E_STEP"]
(NMPC_OK, NMPC_E_ARG, NMPC_E_PATTERN, NMPC_E_ALLOC, NMPC_E_CUDA, NMPC_E_STATE, NMPC_E_NOT_SPD, NMPC_E_INERTIA,
 NMPC_E_MAXITER, NMPC_E_STEP) = range(10)
MODEL_NONE, MODEL_VDP, MODEL_DISTILL, MODEL_PLATE = 0, 1, 2, 3
ORDER_AUTO, ORDER_NATURAL, ORDER_AMD, ORDER_ND, ORDER_TIME_ND = 0, 1, 2, 3, 4

c_i32, c_i64, c_dbl, c_vp = C.c_int32, C.c_int64, C.c_double, C.c_void_p


class nmpc_pattern(C.Structure):
    _fields_ = [("n", c_i64), ("nnz", c_i64), ("rowptr", c_vp), ("colind", c_vp)]


class nmpc_ocp(C.Structure):
    _fields_ = [("model", c_i32), ("N", c_i32), ("nx", c_i32), ("nu", c_i32), ("nr", c_i32), ("dt", c_dbl),
                ("model_params", c_vp), ("n_model_params", c_i32), ("lb", c_vp), ("ub", c_vp), ("u_init", c_vp),
                ("n_g", c_i64), ("g_rowptr", c_vp), ("g_colind", c_vp), ("g_val", c_vp), ("g_lo", c_vp), ("g_hi", c_vp)]


class nmpc_options(C.Structure):
    _fields_ = ([("ordering", c_i32), ("nd_leaf", c_i32), ("relax_small", c_i32), ("relax_zeros", c_dbl),
                 ("smem_front_max", c_i32), ("use_graph", c_i32)]
                + [(k, c_dbl) for k in ("gamma", "eps_outer", "mu0", "mu_warm", "kappa_eps", "kappa_mu", "theta_mu",
                                        "tau_min", "kappa_push", "s_floor", "s_max")]
                + [("max_iter", c_i32)]
                + [(k, c_dbl) for k in ("eta_first", "eta_grow_first", "eta_grow", "eta_shrink", "eta_min", "eta_max",
                                        "warm_push")]
                + [("time_phases", c_i32), ("refine_steps", c_i32), ("globalization", c_i32)]
                + [(k, c_dbl) for k in ("gamma_theta", "gamma_phi", "delta_sw", "s_theta", "s_phi", "eta_phi", "theta_max_fact",
                                        "theta_min_fact")]
                + [("ls_max_backtracks", c_i32), ("grid_limit", c_i32), ("epoch_limit", c_i32)]
                + [("gamma_h", c_dbl), ("cg_tol", c_dbl), ("cg_max_iter", c_i32), ("fuse_rhs", c_i32)])


class nmpc_sym_info(C.Structure):
    _fields_ = ([("n", c_i64), ("nnz_K", c_i64), ("nnz_L", c_i64), ("panel_doubles", c_i64), ("update_doubles", c_i64),
                 ("flops", c_dbl), ("nsuper", c_i32), ("nlevels", c_i32), ("max_front", c_i32), ("max_width", c_i32),
                 ("n_large_fronts", c_i32), ("ordering_used", c_i32), ("analyze_ms", c_dbl)]
                + [(k, c_vp) for k in ("perm", "super_start", "rows_ptr", "rows", "super_parent", "super_level",
                                       "etree_parent")]
                + [("fused_rhs", c_i32)])


class nmpc_stats(C.Structure):
    _fields_ = ([("status", c_i32), ("iters", c_i32), ("factorizations", c_i32), ("eta_retries", c_i32)]
                + [(k, c_dbl) for k in ("E0", "mu", "eta_last", "objective", "ms_total", "ms_eval", "ms_assemble",
                                        "ms_factor", "ms_solve", "ms_vector")])


class nmpc_trace_row(C.Structure):
    _fields_ = [(k, c_dbl) for k in ("mu", "E0", "Emu", "eta", "alpha_pr", "alpha_du", "backtracks", "ms_iter", "ms_eval", "ms_assemble",
                                     "ms_factor", "ms_solve", "ms_vector")]


# every symbol include/nmpc.h declares: name -> (restype, argtypes)
P = C.POINTER
SIGNATURES = {
    "nmpc_default_options": (None, [P(nmpc_options)]),
    "nmpc_symbolic_analyze": (c_i32, [P(nmpc_pattern), P(nmpc_ocp), P(nmpc_options), P(c_vp)]),
    "nmpc_symbolic_info": (c_i32, [c_vp, P(nmpc_sym_info)]),
    "nmpc_symbolic_pattern": (c_i32, [c_vp, P(c_i64), c_vp, c_vp]),
    "nmpc_symbolic_kmap": (c_i32, [c_vp, c_vp, c_vp]),
    "nmpc_symbolic_destroy": (None, [c_vp]),
    "nmpc_analyze": (c_i32, [P(nmpc_pattern), P(nmpc_ocp), P(nmpc_options), c_vp, P(c_vp)]),
    "nmpc_update_params": (c_i32, [c_vp, c_vp, c_vp]),
    "nmpc_update_params_host": (c_i32, [c_vp, c_vp, c_vp]),
    "nmpc_factor": (c_i32, [c_vp, c_vp, c_dbl, P(c_i64)]),
    "nmpc_solve": (c_i32, [c_vp, c_vp, c_i32]),
    "nmpc_factor_rhs": (c_i32, [c_vp, c_vp, c_vp, c_dbl, P(c_i64)]),
    "nmpc_solve_fused": (c_i32, [c_vp, c_vp]),
    "nmpc_solve_static": (c_i32, [c_vp, c_vp, c_vp]),
    "nmpc_kkt_multiply": (c_i32, [c_vp, c_vp, c_vp]),
    "nmpc_ipm_solve": (c_i32, [c_vp, c_i32, c_i32, c_vp, P(nmpc_stats), c_vp, c_i32]),
    "nmpc_hykkt_solve": (c_i32, [c_vp, c_i32, c_i32, c_vp, P(nmpc_stats), c_vp, c_i32]),
    "nmpc_ipm_solve_host": (c_i32, [c_vp, c_i32, c_vp, c_vp, c_vp, P(nmpc_stats)]),
    "nmpc_ipm_solve_batch": (c_i32, [c_vp, c_i32, c_vp, c_vp, c_vp]),
    "nmpc_get_iterate": (c_i32, [c_vp] * 8),
    "nmpc_set_iterate": (c_i32, [c_vp] * 8),
    "nmpc_model_eval": (c_i32, [c_vp] * 7),
    "nmpc_assemble": (c_i32, [c_vp, c_vp, c_vp, c_vp, c_vp, c_dbl, c_vp]),
    "nmpc_get_jac_pattern": (c_i32, [c_vp, P(c_i64), c_vp, c_vp]),
    "nmpc_get_hess_pattern": (c_i32, [c_vp, P(c_i64), c_vp, c_vp]),
    "nmpc_get_kkt_pattern": (c_i32, [c_vp, P(c_i64), c_vp, c_vp]),
    "nmpc_get_info": (c_i32, [c_vp, P(nmpc_sym_info)]),
    "nmpc_get_factor": (c_i32, [c_vp, c_vp]),
    "nmpc_launch_count": (c_i64, [c_vp]),
    "nmpc_last_error": (C.c_char_p, [c_vp]),
    "nmpc_destroy": (None, [c_vp]),
}

# the two extra symbols of include/nmpc_aids.h (measurement build, libnmpc_b200_aids.so)
AIDS_SIGNATURES = {
    "nmpc_fp64_peak": (c_i32, [c_i32, c_i32, P(c_dbl), P(c_dbl)]),
    "nmpc_tile_gemm_peak": (c_i32, [c_i32, c_i32, P(c_dbl), P(c_dbl)]),
    "nmpc_get_task_trace": (c_i64, [c_vp, c_i32, c_vp, c_vp, c_i64]),
}
AIDS_LIB_PATH = os.path.join(_HERE, "libnmpc_b200_aids.so")

_lib = None
_aids = None


def _load(path, signatures):
    if not os.path.exists(path):
        raise RuntimeError(f"{path} is missing: run `python -m paper_2606_04725_b200._build` "
                           "(or __graft_entry__.build()).  There is no CPU fallback.")
    lib = C.CDLL(path)
    for name, (res, args) in signatures.items():
        fn = getattr(lib, name)              # AttributeError if the library does not export a declared symbol
        fn.restype, fn.argtypes = res, args
    return lib


def load_library() -> C.CDLL:
    """Load libnmpc_b200.so (built by paper_2606_04725_b200/_build.py).  Raises if it is missing: no fallback."""
    global _lib
    if _lib is None:
        _lib = _load(LIB_PATH, SIGNATURES)
    return _lib


def load_aids_library() -> C.CDLL:
    """Load libnmpc_b200_aids.so: the measurement build (per-task timestamps, fp64 peak microbenchmarks) of
    include/nmpc_aids.h.  Used by bench.py's live-peak line and by profiling runs, never by the product path."""
    global _aids
    if _aids is None:
        _aids = _load(AIDS_LIB_PATH, {**SIGNATURES, **AIDS_SIGNATURES})
    return _aids


def ipm_solve_batch(handles, warm, ys, check=True):
    """nmpc_ipm_solve_batch: `handles` (each on its own stream) solved concurrently; warm: list of flags; ys: list of DEVICE
    tensors (n doubles each) or None.  Returns the list of nmpc_stats dicts."""
    lib = load_library()
    n = len(handles)
    harr = (c_vp * n)(*[h._h for h in handles])
    warr = (c_i32 * n)(*[int(w) for w in warm])
    yarr = (c_vp * n)(*[_ptr(y) for y in ys]) if ys is not None else None
    stats = (nmpc_stats * n)()
    st = lib.nmpc_ipm_solve_batch(C.cast(harr, c_vp), n, C.cast(warr, c_vp), C.cast(yarr, c_vp) if yarr is not None else None,
                                  C.cast(stats, c_vp))
    if st and (check or st not in (NMPC_E_MAXITER, NMPC_E_INERTIA, NMPC_E_STEP)):
        raise NmpcError(st, "nmpc_ipm_solve_batch")
    return [{k: getattr(stats[i], k) for k, _ in nmpc_stats._fields_} for i in range(n)]


class NmpcError(RuntimeError):
    def __init__(self, status, where, detail=""):
        super().__init__(f"{where}: NMPC_{STATUS_NAMES[status]}" + (f" ({detail})" if detail else ""))
        self.status = status


def _ptr(a):
    """Address of a numpy array (HOST) or torch tensor (HOST or DEVICE) or None."""
    if a is None:
        return None
    if isinstance(a, np.ndarray):
        return a.ctypes.data
    return a.data_ptr()


def default_options(**kw) -> nmpc_options:
    o = nmpc_options()
    load_library().nmpc_default_options(C.byref(o))
    for k, v in kw.items():
        if not hasattr(o, k):
            raise TypeError(f"unknown option {k}")
        setattr(o, k, v)
    return o


def make_ocp(cfg):
    """Marshal an ocp_inputs.OCPConfig-like record into an nmpc_ocp (keeps the numpy buffers alive)."""
    keep = dict(mp=np.ascontiguousarray(cfg.model_params, dtype=np.float64),
                lb=np.ascontiguousarray(cfg.lb, dtype=np.float64), ub=np.ascontiguousarray(cfg.ub, dtype=np.float64),
                ui=np.ascontiguousarray(cfg.u_init, dtype=np.float64))
    g = getattr(cfg, "g_rows", None)
    if g is not None:                                       # general linear rows lo <= G y <= hi (include/nmpc.h)
        keep.update(grp=np.ascontiguousarray(g["rowptr"], dtype=np.int64), gci=np.ascontiguousarray(g["colind"], dtype=np.int32),
                    gv=np.ascontiguousarray(g["val"], dtype=np.float64), glo=np.ascontiguousarray(g["lo"], dtype=np.float64),
                    ghi=np.ascontiguousarray(g["hi"], dtype=np.float64))
    gargs = ((len(keep["glo"]), keep["grp"].ctypes.data, keep["gci"].ctypes.data, keep["gv"].ctypes.data, keep["glo"].ctypes.data,
              keep["ghi"].ctypes.data) if g is not None else (0, None, None, None, None, None))
    o = nmpc_ocp(cfg.model, cfg.N, cfg.nx, cfg.nu, cfg.nr, cfg.dt, keep["mp"].ctypes.data, len(keep["mp"]),
                 keep["lb"].ctypes.data, keep["ub"].ctypes.data, keep["ui"].ctypes.data, *gargs)
    o._keep = keep
    return o


def make_pattern(n, rowptr, colind):
    keep = dict(rp=np.ascontiguousarray(rowptr, dtype=np.int64), ci=np.ascontiguousarray(colind, dtype=np.int32))
    p = nmpc_pattern(n, int(keep["rp"][-1]), keep["rp"].ctypes.data, keep["ci"].ctypes.data)
    p._keep = keep
    return p


def _info_dict(info: nmpc_sym_info, copy_arrays=True):
    d = {k: getattr(info, k) for k, _ in nmpc_sym_info._fields_[:13]}
    d["fused_rhs"] = info.fused_rhs
    if copy_arrays:
        def arr(ptr, count, ct):
            return np.ctypeslib.as_array(C.cast(ptr, P(ct)), shape=(count,)).copy()
        ns, n = info.nsuper, info.n
        d["perm"] = arr(info.perm, n, c_i32)
        d["super_start"] = arr(info.super_start, ns + 1, c_i32)
        d["rows_ptr"] = arr(info.rows_ptr, ns + 1, c_i64)
        d["rows"] = arr(info.rows, int(d["rows_ptr"][-1]), c_i32)
        d["super_parent"] = arr(info.super_parent, ns, c_i32)
        d["super_level"] = arr(info.super_level, ns, c_i32)
        d["etree_parent"] = arr(info.etree_parent, n, c_i32)
    return d


def _get_pattern(fn, h):
    nnz = c_i64()
    st = fn(h, C.byref(nnz), None, None)
    if st:
        raise NmpcError(st, fn.__name__)
    return nnz.value


def fp64_peak(kind: int, repeats: int = 5):
    """nmpc_fp64_peak: (TFLOP/s, ms) of the DFMA (kind 0) / DMMA (kind 1) microbenchmark on the current device."""
    tf, ms = c_dbl(), c_dbl()
    st = load_aids_library().nmpc_fp64_peak(kind, repeats, C.byref(tf), C.byref(ms))
    if st:
        raise NmpcError(st, "nmpc_fp64_peak")
    return tf.value, ms.value


def tile_gemm_peak(K: int = 2048, repeats: int = 3):
    """nmpc_tile_gemm_peak: (TFLOP/s, ms) of the factorization's tile GEMM loop in isolation."""
    tf, ms = c_dbl(), c_dbl()
    st = load_aids_library().nmpc_tile_gemm_peak(K, repeats, C.byref(tf), C.byref(ms))
    if st:
        raise NmpcError(st, "nmpc_tile_gemm_peak")
    return tf.value, ms.value


class Symbolic:
    """Host-only symbolic analysis (nmpc_symbolic_*): usable without a GPU."""

    def __init__(self, pattern=None, ocp=None, options=None):
        self.lib = load_library()
        self._h = c_vp()
        self._keep = (pattern, ocp, options)
        st = self.lib.nmpc_symbolic_analyze(C.byref(pattern) if pattern is not None else None,
                                            C.byref(ocp) if ocp is not None else None,
                                            C.byref(options) if options is not None else None, C.byref(self._h))
        if st:
            raise NmpcError(st, "nmpc_symbolic_analyze")

    def info(self):
        info = nmpc_sym_info()
        self.lib.nmpc_symbolic_info(self._h, C.byref(info))
        return _info_dict(info)

    def pattern(self):
        nnz = _get_pattern(self.lib.nmpc_symbolic_pattern, self._h)
        n = self.info()["n"]
        rp, ci = np.empty(n + 1, np.int64), np.empty(nnz, np.int32)
        self.lib.nmpc_symbolic_pattern(self._h, C.byref(c_i64()), rp.ctypes.data, ci.ctypes.data)
        return rp, ci

    def kmap(self):
        nnz = _get_pattern(self.lib.nmpc_symbolic_pattern, self._h)
        sn, off = np.empty(nnz, np.int32), np.empty(nnz, np.int64)
        self.lib.nmpc_symbolic_kmap(self._h, sn.ctypes.data, off.ctypes.data)
        return sn, off

    def close(self):
        if self._h:
            self.lib.nmpc_symbolic_destroy(self._h)
            self._h = c_vp()

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass


class Handle:
    """nmpc_handle: one OCP structure <-> one CUDA stream.  Methods carry the names of the C entry points."""

    def __init__(self, pattern=None, ocp=None, options=None, stream=None, aids=False):
        self.lib = load_aids_library() if aids else load_library()      # aids=True: measurement build (task traces)
        self._h = c_vp()
        self._keep = (pattern, ocp, options)
        st = self.lib.nmpc_analyze(C.byref(pattern) if pattern is not None else None,
                                   C.byref(ocp) if ocp is not None else None,
                                   C.byref(options) if options is not None else None,
                                   c_vp(stream) if stream else None, C.byref(self._h))
        if st:
            raise NmpcError(st, "nmpc_analyze", (self.lib.nmpc_last_error(None) or b"").decode())

    def _ck(self, st, where, allow=()):
        if st and st not in allow:
            raise NmpcError(st, where, (self.lib.nmpc_last_error(self._h) or b"").decode())
        return st

    def get_info(self):
        info = nmpc_sym_info()
        self._ck(self.lib.nmpc_get_info(self._h, C.byref(info)), "nmpc_get_info")
        return _info_dict(info)

    def update_params(self, x0_dev, ref_dev):
        self._ck(self.lib.nmpc_update_params(self._h, _ptr(x0_dev), _ptr(ref_dev)), "nmpc_update_params")

    def update_params_host(self, x0_host, ref_host):
        self._ck(self.lib.nmpc_update_params_host(self._h, _ptr(x0_host), _ptr(ref_host)), "nmpc_update_params_host")

    def factor(self, values_dev, eta=0.0, check=True):
        info = c_i64(-1)
        st = self.lib.nmpc_factor(self._h, _ptr(values_dev), float(eta), C.byref(info))
        self._ck(st, "nmpc_factor", allow=() if check else (NMPC_E_NOT_SPD,))
        return st, info.value

    def solve(self, rhs_inout_dev, nrhs=1):
        self._ck(self.lib.nmpc_solve(self._h, _ptr(rhs_inout_dev), nrhs), "nmpc_solve")

    def factor_rhs(self, values_dev, rhs_dev, eta=0.0, check=True):
        info = c_i64(-1)
        st = self.lib.nmpc_factor_rhs(self._h, _ptr(values_dev), _ptr(rhs_dev), float(eta), C.byref(info))
        self._ck(st, "nmpc_factor_rhs", allow=() if check else (NMPC_E_NOT_SPD,))
        return st, info.value

    def solve_fused(self, out_dev):
        self._ck(self.lib.nmpc_solve_fused(self._h, _ptr(out_dev)), "nmpc_solve_fused")

    def solve_static(self, rhs_dev, out_dev, check=True):
        """nmpc_solve_static: the two-sided solve with its work vector in the library's static device array (no allocation)."""
        st = self.lib.nmpc_solve_static(self._h, _ptr(rhs_dev), _ptr(out_dev))
        if check:
            self._ck(st, "nmpc_solve_static")
        return st

    def kkt_multiply(self, x_dev, y_dev):
        self._ck(self.lib.nmpc_kkt_multiply(self._h, _ptr(x_dev), _ptr(y_dev)), "nmpc_kkt_multiply")

    def ipm_solve(self, warm, y_inout_dev=None, use_y0=False, trace_cap=0, check=True, _fn="nmpc_ipm_solve"):
        stats = nmpc_stats()
        trace = (nmpc_trace_row * trace_cap)() if trace_cap else None
        st = getattr(self.lib, _fn)(self._h, int(warm), int(use_y0), _ptr(y_inout_dev), C.byref(stats),
                                    C.cast(trace, c_vp) if trace_cap else None, trace_cap)
        self._ck(st, _fn, allow=() if check else (NMPC_E_MAXITER, NMPC_E_INERTIA, NMPC_E_STEP))
        out = {k: getattr(stats, k) for k, _ in nmpc_stats._fields_}
        if trace_cap:
            out["trace"] = [{k: getattr(trace[i], k) for k, _ in nmpc_trace_row._fields_}
                            for i in range(min(trace_cap, stats.iters))]
        return out

    def hykkt_solve(self, warm, y_inout_dev=None, use_y0=False, trace_cap=0, check=True):
        return self.ipm_solve(warm, y_inout_dev, use_y0, trace_cap, check, _fn="nmpc_hykkt_solve")

    def ipm_solve_host(self, warm, x0_host, ref_host, y_out_host, check=True):
        stats = nmpc_stats()
        st = self.lib.nmpc_ipm_solve_host(self._h, int(warm), _ptr(x0_host), _ptr(ref_host), _ptr(y_out_host),
                                          C.byref(stats))
        self._ck(st, "nmpc_ipm_solve_host", allow=() if check else (NMPC_E_MAXITER, NMPC_E_INERTIA, NMPC_E_STEP))
        return {k: getattr(stats, k) for k, _ in nmpc_stats._fields_}

    def get_iterate(self, y=None, sp=None, sm=None, wp=None, wm=None, zL=None, zU=None):
        self._ck(self.lib.nmpc_get_iterate(self._h, *[_ptr(a) for a in (y, sp, sm, wp, wm, zL, zU)]), "nmpc_get_iterate")

    def set_iterate(self, y, sp, sm, wp, wm, zL, zU):
        self._ck(self.lib.nmpc_set_iterate(self._h, *[_ptr(a) for a in (y, sp, sm, wp, wm, zL, zU)]), "nmpc_set_iterate")

    def model_eval(self, y, lam=None, c=None, gradf=None, Jval=None, Wval=None):
        self._ck(self.lib.nmpc_model_eval(self._h, _ptr(y), _ptr(lam), _ptr(c), _ptr(gradf), _ptr(Jval), _ptr(Wval)),
                 "nmpc_model_eval")

    def assemble(self, Jval, Wval, sigma_x, q, eta, Kval):
        self._ck(self.lib.nmpc_assemble(self._h, _ptr(Jval), _ptr(Wval), _ptr(sigma_x), _ptr(q), float(eta), _ptr(Kval)),
                 "nmpc_assemble")

    def _pattern(self, fn, nrows):
        nnz = _get_pattern(fn, self._h)
        rp, ci = np.empty(nrows + 1, np.int64), np.empty(nnz, np.int32)
        self._ck(fn(self._h, C.byref(c_i64()), rp.ctypes.data, ci.ctypes.data), fn.__name__)
        return rp, ci

    def get_jac_pattern(self, m):
        return self._pattern(self.lib.nmpc_get_jac_pattern, m)

    def get_hess_pattern(self, n):
        return self._pattern(self.lib.nmpc_get_hess_pattern, n)

    def get_kkt_pattern(self, n):
        return self._pattern(self.lib.nmpc_get_kkt_pattern, n)

    def get_factor(self):
        info = self.get_info()
        out = np.empty(info["panel_doubles"], np.float64)
        self._ck(self.lib.nmpc_get_factor(self._h, out.ctypes.data), "nmpc_get_factor")
        return out

    def get_task_trace(self, kind):
        """nmpc_get_task_trace (handles created with aids=True): (tasks[nt,4] int32, stamps[nt,8] uint64) of the last
        factorization (0) / solve (1)."""
        nt = int(self.lib.nmpc_get_task_trace(self._h, kind, None, None, 0))
        tasks, stamps = np.zeros((max(nt, 0), 4), np.int32), np.zeros((max(nt, 0), 8), np.uint64)
        if nt > 0:
            self.lib.nmpc_get_task_trace(self._h, kind, tasks.ctypes.data, stamps.ctypes.data, nt)
        return tasks, stamps

    def launch_count(self):
        return int(self.lib.nmpc_launch_count(self._h))

    def close(self):
        if self._h:
            self.lib.nmpc_destroy(self._h)
            self._h = c_vp()

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass
