"""ctypes binding of include/ptefit.h.  Same names as the C ABI; torch is used only for device
memory and streams."""
import ctypes as C
import os

import numpy as np

HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(HERE, "libptefit.so")

EXPORTED_SYMBOLS = [
    "ptefit_create", "ptefit_reconstruct", "ptefit_reconstruct_host", "ptefit_destroy", "ptefit_last_error",
    "ptefit_global_error", "ptefit_debug_gs_solve", "ptefit_debug_search", "ptefit_debug_fit",
    "ptefit_last_launch_count", "ptefit_set_profiling", "ptefit_get_stage_ms", "ptefit_greens_table", "ptefit_get_coil_currents", "ptefit_flux_surfaces",
    "ptefit_gs_solve_noalloc",
]

PTEFIT_FP32, PTEFIT_FP64 = 0, 1
GEMM_3XTF32, GEMM_FFMA = 0, 2
OPT_NO_GRAPH, OPT_NO_FUSED_BASIS, OPT_SOLVE_FFMA = 1, 2, 4
FAMILY_POLY, FAMILY_SPLINE = 0, 1
NOALLOC_SCRATCH_BYTES = 8 << 20   # PTEFIT_NOALLOC_SCRATCH_BYTES of include/ptefit.h


class PtefitError(RuntimeError):
    pass


class _Grid(C.Structure):
    _fields_ = [("nr", C.c_int), ("nz", C.c_int), ("rmin", C.c_double), ("rmax", C.c_double),
                ("zmin", C.c_double), ("zmax", C.c_double)]


class _Geometry(C.Structure):
    _fields_ = [("n_meas", C.c_int), ("n_coil", C.c_int), ("sigma", C.c_void_p), ("n_lim", C.c_int),
                ("lim_r", C.c_void_p), ("lim_z", C.c_void_p), ("lim_mask", C.c_void_p), ("xpt_mask", C.c_void_p),
                ("ip_sign", C.c_int), ("cold_rc", C.c_double), ("cold_zc", C.c_double), ("cold_a", C.c_double),
                ("cold_b", C.c_double)]


class _Tables(C.Structure):
    _fields_ = [("gp", C.c_void_p), ("gc", C.c_void_p), ("gb", C.c_void_p), ("ggc", C.c_void_p)]


class _Term(C.Structure):
    _fields_ = [("kind", C.c_int), ("family", C.c_int), ("i", C.c_int), ("N", C.c_int), ("n_knots", C.c_int),
                ("knots", C.c_void_p), ("tension", C.c_double)]


class _Basis(C.Structure):
    _fields_ = [("n_terms", C.c_int), ("terms", C.POINTER(_Term)), ("lambda_reg", C.c_double), ("relax", C.c_double),
                ("lsq_method", C.c_int), ("fit_coils", C.c_int), ("sigma_ic", C.c_void_p)]


class _ProfileSpec(C.Structure):
    _fields_ = [("n_prof", C.c_int), ("n_chord", C.c_int), ("n_bisect", C.c_int), ("n_q", C.c_int), ("mu", C.c_void_p),
                ("nu", C.c_void_p), ("f_vac", C.c_double)]


class _Options(C.Structure):
    _fields_ = [("precision", C.c_int), ("gemm", C.c_int), ("max_batch", C.c_int), ("flags", C.c_int), ("tc_split_k", C.c_int)]


_lib = None


def load_library():
    """dlopen libptefit.so (built in-tree by build.py); fails loudly if it is missing."""
    global _lib
    if _lib is None:
        if not os.path.exists(LIB_PATH):
            raise PtefitError(f"{LIB_PATH} is missing: run `python -m paper_2601_12378_b200.build` "
                              "(there is no fallback path)")
        lib = C.CDLL(LIB_PATH)
        lib.ptefit_create.restype = C.c_int
        lib.ptefit_create.argtypes = [C.c_void_p] * 5 + [C.POINTER(C.c_void_p)]
        lib.ptefit_reconstruct.restype = C.c_int
        lib.ptefit_reconstruct.argtypes = ([C.c_void_p, C.c_int, C.c_void_p, C.c_void_p, C.c_int, C.c_int]
                                           + [C.c_void_p] * 11)
        lib.ptefit_reconstruct_host.restype = C.c_int
        lib.ptefit_reconstruct_host.argtypes = ([C.c_void_p, C.c_int, C.c_void_p, C.c_void_p, C.c_int, C.c_int]
                                                + [C.c_void_p] * 10)
        lib.ptefit_destroy.restype = None
        lib.ptefit_destroy.argtypes = [C.c_void_p]
        lib.ptefit_last_error.restype = C.c_char_p
        lib.ptefit_last_error.argtypes = [C.c_void_p]
        lib.ptefit_global_error.restype = C.c_char_p
        lib.ptefit_debug_gs_solve.restype = C.c_int
        lib.ptefit_debug_gs_solve.argtypes = [C.c_void_p, C.c_int] + [C.c_void_p] * 4
        lib.ptefit_gs_solve_noalloc.restype = C.c_int
        lib.ptefit_gs_solve_noalloc.argtypes = [C.c_void_p, C.c_int] + [C.c_void_p] * 4
        lib.ptefit_debug_search.restype = C.c_int
        lib.ptefit_debug_search.argtypes = [C.c_void_p, C.c_int] + [C.c_void_p] * 10
        lib.ptefit_debug_fit.restype = C.c_int
        lib.ptefit_debug_fit.argtypes = [C.c_void_p, C.c_int] + [C.c_void_p] * 9
        lib.ptefit_last_launch_count.restype = C.c_int
        lib.ptefit_last_launch_count.argtypes = [C.c_void_p]
        lib.ptefit_set_profiling.restype = C.c_int
        lib.ptefit_set_profiling.argtypes = [C.c_void_p, C.c_int]
        lib.ptefit_get_stage_ms.restype = C.c_int
        lib.ptefit_get_stage_ms.argtypes = [C.c_void_p, C.POINTER(C.c_float)]
        lib.ptefit_flux_surfaces.restype = C.c_int
        lib.ptefit_flux_surfaces.argtypes = [C.c_void_p, C.c_int] + [C.c_void_p] * 8
        lib.ptefit_get_coil_currents.restype = C.c_int
        lib.ptefit_get_coil_currents.argtypes = [C.c_void_p, C.c_int, C.c_void_p, C.c_void_p]
        lib.ptefit_greens_table.restype = C.c_int
        lib.ptefit_greens_table.argtypes = ([C.c_int] + [C.c_void_p] * 4 + [C.c_int] + [C.c_void_p] * 4 + [C.c_int, C.c_void_p])
        _lib = lib
    return _lib


def poly_terms(n_p, n_ff, delz=False, spline=None):
    """Eq. 10 term list: P' terms x^i - x^n_p (i < n_p), FF' terms x^j - x^n_ff, optional FF'-type
    tension-spline terms (spline = dict(knots, tension, terms)), optional delz.  Each term is
    (kind, i, N) or (kind, i, N, family, knots, tension)."""
    t = [(0, i, n_p) for i in range(n_p)] + [(1, j, n_ff) for j in range(n_ff)]
    if spline is not None:
        kn = np.ascontiguousarray(spline["knots"], np.float64)
        t += [(1, int(q), 0, FAMILY_SPLINE, kn, float(spline["tension"])) for q in spline["terms"]]
    if delz:
        t.append((2, 0, 0))
    return t


def _term_struct(t, keep):
    if len(t) == 3:
        return _Term(int(t[0]), FAMILY_POLY, int(t[1]), int(t[2]), 0, None, 0.0)
    kind, i, N, fam, kn, tau = t
    kn = np.ascontiguousarray(kn, np.float64)
    keep.append(kn)
    return _Term(int(kind), int(fam), int(i), int(N), len(kn), _ptr(kn), float(tau))


def _f64(a):
    return np.ascontiguousarray(a, dtype=np.float64)


def _ptr(a):
    return a.ctypes.data_as(C.c_void_p) if a is not None else None


def ptefit_create(grid, geom, tables, terms, lambda_reg, relax, precision, gemm, max_batch, flags=0, tc_split_k=0,
                  lsq_method=0, fit_coils=0, sigma_ic=None):
    """Marshal numpy inputs into the C structs and call ptefit_create.  Returns the handle."""
    lib = load_library()
    g = _Grid(int(grid["nr"]), int(grid["nz"]), grid["rmin"], grid["rmax"], grid["zmin"], grid["zmax"])
    keep = dict(sigma=_f64(geom["sigma"]), lim_r=_f64(geom["lim_r"]), lim_z=_f64(geom["lim_z"]),
                lim_mask=np.ascontiguousarray(geom["lim_mask"], dtype=np.uint8).ravel(),
                xpt_mask=None if geom.get("xpt_mask") is None else np.ascontiguousarray(geom["xpt_mask"], dtype=np.uint8).ravel(),
                gp=_f64(tables["gp"]), gc=_f64(tables["gc"]), gb=_f64(tables["gb"]), ggc=_f64(tables["ggc"]))
    ge = _Geometry(int(geom["n_meas"]), int(geom["n_coil"]), _ptr(keep["sigma"]), len(keep["lim_r"]),
                   _ptr(keep["lim_r"]), _ptr(keep["lim_z"]), _ptr(keep["lim_mask"]), _ptr(keep["xpt_mask"]),
                   int(geom.get("ip_sign", 1)), geom["cold_rc"], geom["cold_zc"], geom["cold_a"], geom["cold_b"])
    tb = _Tables(_ptr(keep["gp"]), _ptr(keep["gc"]), _ptr(keep["gb"]), _ptr(keep["ggc"]))
    kk = []
    tarr = (_Term * len(terms))(*[_term_struct(t, kk) for t in terms])
    sic = None if sigma_ic is None else _f64(sigma_ic)
    ba = _Basis(len(terms), tarr, float(lambda_reg), float(relax), int(lsq_method), int(fit_coils), _ptr(sic))
    op = _Options(int(precision), int(gemm), int(max_batch), int(flags), int(tc_split_k))
    h = C.c_void_p()
    st = lib.ptefit_create(C.byref(g), C.byref(ge), C.byref(tb), C.byref(ba), C.byref(op), C.byref(h))
    if st != 0:
        raise PtefitError(f"ptefit_create failed ({st}): {lib.ptefit_global_error().decode()}")
    return h


def ptefit_destroy(h):
    load_library().ptefit_destroy(h)


def _dp(t):
    return C.c_void_p(t.data_ptr()) if t is not None else None


def ptefit_reconstruct(h, batch, d_b, d_ic, n_iter, warm_start, d_psi, d_coeffs, d_axis_ij=None, d_axis_rzpsi=None,
                       d_xpt_ij=None, d_xpt_rzpsi=None, d_psi_bnd=None, d_limited=None, d_chi2=None, d_status=None,
                       stream=None):
    """torch CUDA tensors in, asynchronous on `stream` (torch.cuda.Stream or None = current)."""
    import torch
    lib = load_library()
    s = stream if stream is not None else torch.cuda.current_stream()
    st = lib.ptefit_reconstruct(h, batch, _dp(d_b), _dp(d_ic), n_iter, int(warm_start), _dp(d_psi), _dp(d_coeffs),
                                _dp(d_axis_ij), _dp(d_axis_rzpsi), _dp(d_xpt_ij), _dp(d_xpt_rzpsi), _dp(d_psi_bnd),
                                _dp(d_limited), _dp(d_chi2), _dp(d_status), C.c_void_p(s.cuda_stream))
    if st != 0:
        raise PtefitError(f"ptefit_reconstruct failed ({st}): {lib.ptefit_last_error(h).decode()}")


class Reconstructor:
    """Convenience owner of a handle plus output tensors (argument marshalling only)."""

    def __init__(self, dev, precision="fp32", gemm=GEMM_3XTF32, max_batch=1, delz=None, lambda_reg=None, relax=None,
                 flags=0, tc_split_k=0, lsq_method=0, fit_coils=0, sigma_ic=None):
        import torch
        if not torch.cuda.is_available():
            raise PtefitError("no CUDA device: the PTEFIT hot path has no CPU fallback")
        self.torch = torch
        b = dev["basis"]
        self.delz = bool(b.get("delz", 0)) if delz is None else bool(delz)
        self.terms = poly_terms(b["n_p"], b["n_ff"], self.delz, b.get("spline"))
        self.prec = PTEFIT_FP32 if precision == "fp32" else PTEFIT_FP64
        self.dtype = torch.float32 if precision == "fp32" else torch.float64
        self.npdtype = np.float32 if precision == "fp32" else np.float64
        self.grid = dev["grid"]
        self.nr, self.nz = dev["grid"]["nr"], dev["grid"]["nz"]
        self.M, self.nc = dev["geom"]["n_meas"], dev["geom"]["n_coil"]
        self.nt = len(self.terms)
        self.max_batch = max_batch
        self.h = ptefit_create(dev["grid"], dev["geom"], dev["tables"], self.terms,
                               b.get("lambda_reg", 0.0) if lambda_reg is None else lambda_reg,
                               b.get("relax", 1.0) if relax is None else relax, self.prec, gemm, max_batch, flags, tc_split_k,
                               lsq_method, fit_coils, sigma_ic)
        self.lib = load_library()
        self._alloc(max_batch)

    def _alloc(self, B):
        t, dt = self.torch, self.dtype
        kw = dict(device="cuda")
        self.psi = t.zeros(B, self.nz, self.nr, dtype=dt, **kw)
        self.coeffs = t.zeros(B, self.nt, dtype=dt, **kw)
        self.axis_ij = t.zeros(B, 2, dtype=t.int32, **kw)
        self.axis_rzpsi = t.zeros(B, 3, dtype=dt, **kw)
        self.xpt_ij = t.zeros(B, 2, dtype=t.int32, **kw)
        self.xpt_rzpsi = t.zeros(B, 3, dtype=dt, **kw)
        self.psi_bnd = t.zeros(B, dtype=dt, **kw)
        self.limited = t.zeros(B, dtype=t.int32, **kw)
        self.chi2 = t.zeros(B, dtype=dt, **kw)
        self.status = t.zeros(B, dtype=t.int32, **kw)

    def reconstruct(self, d_b, d_ic, n_iter, warm_start=False, stream=None):
        B = d_b.shape[0]
        ptefit_reconstruct(self.h, B, d_b, d_ic, n_iter, warm_start, self.psi, self.coeffs, self.axis_ij,
                           self.axis_rzpsi, self.xpt_ij, self.xpt_rzpsi, self.psi_bnd, self.limited, self.chi2,
                           self.status, stream)

    def reconstruct_host(self, b, ic, n_iter, out, warm_start=False):
        """HOST numpy buffers in and out (dict `out` of preallocated arrays) via ptefit_reconstruct_host."""
        B = b.shape[0]
        st = self.lib.ptefit_reconstruct_host(self.h, B, _ptr(b), _ptr(ic), n_iter, int(warm_start), _ptr(out["psi"]),
                                              _ptr(out["coeffs"]), _ptr(out.get("axis_ij")), _ptr(out.get("axis_rzpsi")),
                                              _ptr(out.get("xpt_ij")), _ptr(out.get("xpt_rzpsi")), _ptr(out.get("psi_bnd")),
                                              _ptr(out.get("limited")), _ptr(out.get("chi2")), _ptr(out.get("status")))
        if st != 0:
            raise PtefitError(f"ptefit_reconstruct_host failed ({st}): {self.lib.ptefit_last_error(self.h).decode()}")

    def host_outputs(self, B):
        f = self.npdtype
        return dict(psi=np.zeros((B, self.nz, self.nr), f), coeffs=np.zeros((B, self.nt), f),
                    axis_ij=np.zeros((B, 2), np.int32), axis_rzpsi=np.zeros((B, 3), f), xpt_ij=np.zeros((B, 2), np.int32),
                    xpt_rzpsi=np.zeros((B, 3), f), psi_bnd=np.zeros(B, f), limited=np.zeros(B, np.int32),
                    chi2=np.zeros(B, f), status=np.zeros(B, np.int32))

    def _call(self, fn, *args):
        st = fn(self.h, *args)
        if st != 0:
            raise PtefitError(f"{fn.__name__} failed ({st}): {self.lib.ptefit_last_error(self.h).decode()}")

    def debug_gs_solve(self, d_I, d_pbd, d_psi_out):
        s = self.torch.cuda.current_stream()
        self._call(self.lib.ptefit_debug_gs_solve, d_I.shape[0], _dp(d_I), _dp(d_pbd), _dp(d_psi_out), C.c_void_p(s.cuda_stream))

    def gs_solve_noalloc(self, d_I, d_pbd, d_psi_out):
        """ptefit_gs_solve_noalloc: the Delta* solve with its workspace in the library's static device array
        (FP64 handles; at most NOALLOC_SCRATCH_BYTES of workspace per call; no allocation inside the call)."""
        s = self.torch.cuda.current_stream()
        self._call(self.lib.ptefit_gs_solve_noalloc, d_I.shape[0], _dp(d_I), _dp(d_pbd), _dp(d_psi_out), C.c_void_p(s.cuda_stream))

    def debug_search(self, d_psi, d_xn):
        s = self.torch.cuda.current_stream()
        self._call(self.lib.ptefit_debug_search, d_psi.shape[0], _dp(d_psi), _dp(d_xn), _dp(self.axis_ij), _dp(self.axis_rzpsi),
                   _dp(self.xpt_ij), _dp(self.xpt_rzpsi), _dp(self.psi_bnd), _dp(self.limited), _dp(self.status),
                   C.c_void_p(s.cuda_stream))

    def debug_fit(self, d_xn, d_b, d_ic, d_xprev, d_resp):
        s = self.torch.cuda.current_stream()
        self._call(self.lib.ptefit_debug_fit, d_xn.shape[0], _dp(d_xn), _dp(d_b), _dp(d_ic), _dp(d_xprev), _dp(d_resp),
                   _dp(self.coeffs), _dp(self.chi2), _dp(self.status), C.c_void_p(s.cuda_stream))

    def flux_surfaces(self, B, n_prof=33, n_chord=128, n_bisect=10, munu=((-1, -1), (-1, -2), (0, 0)), f_vac=0.0, want_vert=True):
        """Flux-surface post-processing of the last reconstruct call (ptefit_flux_surfaces).  Returns a dict of
        torch tensors Q[B, n_prof, n_q], q[B, n_prof], geom[B, 6], vert[B, n_prof, n_chord, 2], status[B]."""
        t = self.torch
        mu = np.ascontiguousarray([m for m, _ in munu], np.int32); nu = np.ascontiguousarray([n for _, n in munu], np.int32)
        sp = _ProfileSpec(int(n_prof), int(n_chord), int(n_bisect), len(munu), _ptr(mu), _ptr(nu), float(f_vac))
        kw = dict(dtype=self.dtype, device="cuda")
        out = dict(Q=t.zeros(B, n_prof, len(munu), **kw), q=t.zeros(B, n_prof, **kw), geom=t.zeros(B, 6, **kw),
                   vert=t.zeros(B, n_prof, n_chord, 2, **kw) if want_vert else None, status=t.zeros(B, dtype=t.int32, device="cuda"))
        s = t.cuda.current_stream()
        self._call(self.lib.ptefit_flux_surfaces, B, C.byref(sp), _dp(self.psi), _dp(out["Q"]), _dp(out["q"]), _dp(out["geom"]),
                   _dp(out["vert"]), _dp(out["status"]), C.c_void_p(s.cuda_stream))
        return out

    def coil_currents(self, B):
        """Fitted coil currents of the last call (fit_coils = 1): torch tensor [B, n_coil]."""
        out = self.torch.zeros(B, self.nc, dtype=self.dtype, device="cuda")
        s = self.torch.cuda.current_stream()
        self._call(self.lib.ptefit_get_coil_currents, B, _dp(out), C.c_void_p(s.cuda_stream))
        return out

    def launch_count(self):
        return self.lib.ptefit_last_launch_count(self.h)

    def set_profiling(self, on):
        self.lib.ptefit_set_profiling(self.h, int(on))

    def stage_ms(self):
        out = (C.c_float * 6)()
        self._call(self.lib.ptefit_get_stage_ms, out)
        return dict(zip(("setup", "response", "lsq", "boundary", "solve", "search"), list(out)))

    def close(self):
        if self.h is not None:
            ptefit_destroy(self.h)
            self.h = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass


def ptefit_greens_table(d_fld_r, d_fld_z, d_src_r, d_src_z, d_out, d_fld_cos=None, d_fld_sin=None, d_src_w=None, transpose=False,
                        stream=None):
    """FP64 torch CUDA tensors in; d_out [n_fld, n_src] (or [n_src, n_fld] if transpose) is filled asynchronously."""
    import torch
    lib = load_library()
    s = stream if stream is not None else torch.cuda.current_stream()
    st = lib.ptefit_greens_table(int(d_fld_r.numel()), _dp(d_fld_r), _dp(d_fld_z), _dp(d_fld_cos), _dp(d_fld_sin), int(d_src_r.numel()),
                                 _dp(d_src_r), _dp(d_src_z), _dp(d_src_w), _dp(d_out), int(bool(transpose)), C.c_void_p(s.cuda_stream))
    if st != 0:
        raise PtefitError(f"ptefit_greens_table failed ({st}): {lib.ptefit_global_error().decode()}")


def shard_slices(n_slices, rank, world):
    """Contiguous block of time slices rank `rank` of `world` reconstructs (slices are independent,
    tables are replicated, no data-path collective).  Returns (first, count); earlier ranks take
    the remainder."""
    base, rem = divmod(int(n_slices), int(world))
    count = base + (1 if rank < rem else 0)
    first = rank * base + min(rank, rem)
    return first, count
