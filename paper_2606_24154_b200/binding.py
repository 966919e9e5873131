"""ctypes binding of libneb.so: same names as include/neb.h, marshalling only."""
import ctypes as C
import os
import re

import numpy as np

from . import build as _build

NEB_RECT, NEB_TRI, NEB_WIRE = 0, 1, 2
NEB_BC_DIRICHLET, NEB_BC_DIELECTRIC = 0, 1
NEB_DIST_BLOCK = 256
NEB_EVAL_STATIC_MAX_POINTS = 65536
NEB_OPT_MATH, NEB_OPT_LU_BLOCK, NEB_OPT_PROFILE, NEB_OPT_LU_PANEL, NEB_OPT_LU_LOOKAHEAD, NEB_OPT_EVAL_SPLITS, NEB_OPT_SOLVER, NEB_OPT_PAIR_STRIPS = 0, 1, 2, 3, 4, 5, 6, 7
STAGES = ["geometry", "assemble", "equil", "lu", "lu_gemm", "rhs", "trisolve", "eval", "charges", "reduce", "fastvol"]
_STATUS = {1: "NEB_EINVAL", 2: "NEB_ENOMEM", 3: "NEB_ESTATE", 4: "NEB_ESINGULAR", 5: "NEB_ECUDA"}

_HERE = os.path.dirname(os.path.abspath(__file__))
_HEADER = os.path.join(os.path.dirname(_HERE), "include", "neb.h")
_lib = None


class NebError(RuntimeError):
    def __init__(self, status, msg):
        super().__init__(f"{_STATUS.get(status, status)}: {msg}")
        self.status = status


def lib_path() -> str:
    return _build.LIB


def exported_symbols():
    """Names declared in include/neb.h (every `neb_*(` prototype)."""
    with open(_HEADER) as fh:
        text = fh.read()
    return sorted(set(re.findall(r"\b(neb_[a-z0-9_]+)\s*\(", text)))


def lib():
    """Loads libneb.so (building it in-tree if it is missing); raises if that is impossible."""
    global _lib
    if _lib is None:
        path = _build.build()
        L = C.CDLL(path)
        vp, i32, i64, dbl = C.c_void_p, C.c_int32, C.c_int64, C.c_double
        L.neb_create.argtypes = [C.POINTER(vp), C.c_int, vp]
        L.neb_destroy.argtypes = [vp]
        L.neb_destroy.restype = None
        L.neb_last_error.argtypes = [vp]
        L.neb_last_error.restype = C.c_char_p
        L.neb_set_option.argtypes = [vp, i32, i64]
        L.neb_assemble.argtypes = [vp, i64] + [vp] * 10 + [i32, vp]
        L.neb_solve.argtypes = [vp, vp]
        L.neb_set_sigma.argtypes = [vp, vp]
        L.neb_eval.argtypes = [vp, i64, vp, vp, vp]
        L.neb_eval_static.argtypes = [vp, i64, vp, vp, vp]
        L.neb_add_space_charge.argtypes = [vp, i64, vp, vp, i32]
        L.neb_solve_weighting.argtypes = [vp, vp, vp]
        L.neb_solve_weighting_multi.argtypes = [vp, i32, vp, vp]
        L.neb_set_adaptive.argtypes = [vp, dbl]
        L.neb_voxelize_space_charge.argtypes = [vp, vp, vp, vp, C.POINTER(i64)]
        L.neb_get_line_charges.argtypes = [vp, vp]
        L.neb_fastvol_build.argtypes = [vp, i32, i32, i32, i32, vp, vp, i32]
        L.neb_fastvol_eval.argtypes = [vp, i32, i64, vp, vp, vp]
        L.neb_fastvol_get.argtypes = [vp, i32, vp]
        L.neb_push.argtypes = [vp, i64, vp, vp, dbl]
        L.neb_get_matrix.argtypes = [vp, vp]
        L.neb_get_matrix_rows.argtypes = [vp, i64, vp, vp]
        L.neb_get_rhs.argtypes = [vp, vp]
        L.neb_fp64_peak.argtypes = [vp, i32, C.POINTER(dbl)]
        L.neb_stage_ms.argtypes = [vp, i32, C.POINTER(dbl), C.POINTER(i64)]
        L.neb_get_counter.argtypes = [vp, i32, C.POINTER(dbl)]
        L.neb_reset_stats.argtypes = [vp]
        L.neb_launch_count.argtypes = [vp]
        L.neb_launch_count.restype = i64
        L.neb_set_svd_cutoff.argtypes = [vp, dbl]
        L.neb_get_singular_values.argtypes = [vp, vp, C.POINTER(i32)]
        L.neb_dist_configure.argtypes = [vp, i32, i32]
        L.neb_dist_npad.argtypes = [vp]
        L.neb_dist_npad.restype = i64
        L.neb_dist_row_scales.argtypes = [vp, vp, i32]
        L.neb_dist_factor_block.argtypes = [vp, i64, vp, vp, vp]
        L.neb_dist_apply_block.argtypes = [vp, i64, vp, vp, i32]
        L.neb_dist_finish_factor.argtypes = [vp, C.POINTER(i32)]
        L.neb_dist_rhs.argtypes = [vp, vp]
        L.neb_dist_tri_block.argtypes = [vp, i32, i64, vp, vp]
        L.neb_dist_set_solution.argtypes = [vp, vp, vp]
        _lib = L
    return _lib


def _ptr(a):
    """Raw address of a torch tensor (device or host) or a numpy array; None -> NULL."""
    if a is None:
        return None
    if isinstance(a, np.ndarray):
        return a.ctypes.data
    return a.data_ptr()            # torch.Tensor


def _check_arr(a, dtype_np, dtype_name, count, name):
    if a is None:
        return None
    if isinstance(a, np.ndarray):
        if a.dtype != dtype_np or not a.flags["C_CONTIGUOUS"]:
            a = np.ascontiguousarray(a, dtype=dtype_np)
    else:
        import torch
        want = {"float64": torch.float64, "int32": torch.int32}[dtype_name]
        if a.dtype != want or not a.is_contiguous():
            a = a.to(want).contiguous()
    n = a.size if isinstance(a, np.ndarray) else a.numel()
    if n != count:
        raise ValueError(f"{name}: expected {count} values, got {n}")
    return a


class Neb:
    """One neb_ctx.  Arrays may be numpy arrays (host) or torch tensors (host or cuda); vectors are SoA
    with shape (3, n).  Outputs are returned in the same kind of memory as `pts` unless `out` is given."""

    def __init__(self, device: int = 0, stream=None):
        import torch
        if not torch.cuda.is_available():
            raise NebError(5, "no CUDA device: this library has no CPU path")
        self._L = lib()
        self._h = C.c_void_p()
        if stream is None:
            stream = torch.cuda.current_stream(device).cuda_stream
        self.device = device
        st = self._L.neb_create(C.byref(self._h), device, C.c_void_p(stream))
        if st != 0:
            raise NebError(st, "neb_create failed (needs an sm_100 device)")
        self.n = 0

    def _ck(self, st):
        if st != 0:
            raise NebError(st, self._L.neb_last_error(self._h).decode())

    def close(self):
        if getattr(self, "_h", None) is not None and self._h:
            self._L.neb_destroy(self._h)
            self._h = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def set_option(self, option: int, value: int):
        self._ck(self._L.neb_set_option(self._h, option, value))

    def assemble(self, kind, v0, e1, e2, bc_kind, bc_value=None, radius=None, colloc=None, eps_plus=None,
                 eps_minus=None, img_shift=None):
        n = int(kind.shape[0])
        a = dict(kind=_check_arr(kind, np.int32, "int32", n, "kind"), v0=_check_arr(v0, np.float64, "float64", 3 * n, "v0"),
                 e1=_check_arr(e1, np.float64, "float64", 3 * n, "e1"), e2=_check_arr(e2, np.float64, "float64", 3 * n, "e2"),
                 radius=_check_arr(radius, np.float64, "float64", n, "radius"),
                 colloc=_check_arr(colloc, np.float64, "float64", 3 * n, "colloc"),
                 bc_kind=_check_arr(bc_kind, np.int32, "int32", n, "bc_kind"),
                 bc_value=_check_arr(bc_value, np.float64, "float64", n, "bc_value"),
                 eps_plus=_check_arr(eps_plus, np.float64, "float64", n, "eps_plus"),
                 eps_minus=_check_arr(eps_minus, np.float64, "float64", n, "eps_minus"))
        n_img = 0
        if img_shift is not None:
            n_img = int(img_shift.shape[1])
            img_shift = _check_arr(img_shift, np.float64, "float64", 3 * n_img, "img_shift")
        self._ck(self._L.neb_assemble(self._h, n, _ptr(a["kind"]), _ptr(a["v0"]), _ptr(a["e1"]), _ptr(a["e2"]),
                                      _ptr(a["radius"]), _ptr(a["colloc"]), _ptr(a["bc_kind"]), _ptr(a["bc_value"]),
                                      _ptr(a["eps_plus"]), _ptr(a["eps_minus"]), n_img, _ptr(img_shift)))
        self.n = n

    def assemble_problem(self, pr, colloc=None):
        """Convenience: a workloads.configs.Problem (host arrays)."""
        self.assemble(pr.kind, pr.v0, pr.e1, pr.e2, pr.bc_kind, pr.bc_value, radius=pr.radius, colloc=colloc,
                      eps_plus=pr.eps_plus, eps_minus=pr.eps_minus, img_shift=pr.img_shift)

    def solve(self, out=None):
        """Returns sigma (n) as a numpy array, or fills `out` (numpy or torch, host or device)."""
        if out is None:
            out = np.empty(self.n)
        self._ck(self._L.neb_solve(self._h, _ptr(out)))
        return out

    def solve_resident(self):
        """neb_solve without reading sigma back."""
        self._ck(self._L.neb_solve(self._h, None))

    def set_sigma(self, sigma):
        sigma = _check_arr(sigma, np.float64, "float64", self.n, "sigma")
        self._ck(self._L.neb_set_sigma(self._h, _ptr(sigma)))

    def eval(self, pts, phi=None, E=None, want_phi=True, want_E=True):
        m = int(pts.shape[1])
        pts = _check_arr(pts, np.float64, "float64", 3 * m, "pts")
        if isinstance(pts, np.ndarray):
            if phi is None and want_phi:
                phi = np.empty(m)
            if E is None and want_E:
                E = np.empty((3, m))
        else:
            import torch
            if phi is None and want_phi:
                phi = torch.empty(m, dtype=torch.float64, device=pts.device)
            if E is None and want_E:
                E = torch.empty((3, m), dtype=torch.float64, device=pts.device)
        self._ck(self._L.neb_eval(self._h, m, _ptr(pts), _ptr(phi), _ptr(E)))
        return phi, E

    def eval_static(self, pts, phi, E):
        """neb_eval_static: pts (3, m), phi (m) and E (3, m) are contiguous float64 CUDA tensors supplied by the caller
        (either output may be None); m <= NEB_EVAL_STATIC_MAX_POINTS; nothing is allocated, here or in the library."""
        self._ck(self._L.neb_eval_static(self._h, int(pts.shape[1]), _ptr(pts), _ptr(phi), _ptr(E)))
        return phi, E

    def add_space_charge(self, pos, charge, replace=True):
        q = 0 if charge is None else int(charge.shape[0])
        pos = _check_arr(pos, np.float64, "float64", 3 * q, "pos")
        charge = _check_arr(charge, np.float64, "float64", q, "charge")
        self._ck(self._L.neb_add_space_charge(self._h, q, _ptr(pos), _ptr(charge), 1 if replace else 0))

    def set_adaptive(self, far_distance: float):
        """neb_set_adaptive: image copies at least far_distance (m) away become point charges in eval (0 = off)."""
        self._ck(self._L.neb_set_adaptive(self._h, float(far_distance)))

    def solve_weighting(self, bc_value_w, out=None):
        """neb_solve_weighting: sigma_w (n) for the weighting potentials bc_value_w (n), on the resident factors."""
        bc_value_w = _check_arr(bc_value_w, np.float64, "float64", self.n, "bc_value_w")
        if out is None:
            out = np.empty(self.n)
        self._ck(self._L.neb_solve_weighting(self._h, _ptr(bc_value_w), _ptr(out)))
        return out

    def solve_weighting_multi(self, bc_values_w, out=None):
        """neb_solve_weighting_multi: bc_values_w (n_rhs, n) -> sigma_w (n_rhs, n), one pass per 8 electrodes."""
        n_rhs = int(bc_values_w.shape[0])
        bc_values_w = _check_arr(bc_values_w, np.float64, "float64", n_rhs * self.n, "bc_values_w")
        if out is None:
            out = np.empty((n_rhs, self.n))
        self._ck(self._L.neb_solve_weighting_multi(self._h, n_rhs, _ptr(bc_values_w), _ptr(out)))
        return out

    def fastvol_build(self, slot: int, shape, origin, spacing, with_charges: bool = True):
        """neb_fastvol_build: shape = (nx, ny, nz), origin and spacing 3 floats each (host)."""
        nx, ny, nz = (int(v) for v in shape)
        origin = np.ascontiguousarray(origin, dtype=np.float64)
        spacing = np.ascontiguousarray(spacing, dtype=np.float64)
        if origin.shape != (3,) or spacing.shape != (3,):
            raise ValueError("origin and spacing must hold 3 values")
        self._ck(self._L.neb_fastvol_build(self._h, slot, nx, ny, nz, _ptr(origin), _ptr(spacing), 1 if with_charges else 0))
        self._fv_nodes = getattr(self, "_fv_nodes", {})
        self._fv_nodes[slot] = nx * ny * nz

    def fastvol_eval(self, slot: int, pts, phi=None, E=None):
        m = int(pts.shape[1])
        pts = _check_arr(pts, np.float64, "float64", 3 * m, "pts")
        if isinstance(pts, np.ndarray):
            phi = np.empty(m) if phi is None else phi
            E = np.empty((3, m)) if E is None else E
        else:
            import torch
            phi = torch.empty(m, dtype=torch.float64, device=pts.device) if phi is None else phi
            E = torch.empty((3, m), dtype=torch.float64, device=pts.device) if E is None else E
        self._ck(self._L.neb_fastvol_eval(self._h, slot, m, _ptr(pts), _ptr(phi), _ptr(E)))
        return phi, E

    def fastvol_get(self, slot: int):
        """Node values (4, nx*ny*nz): Phi, Ex, Ey, Ez (test hook)."""
        nn = getattr(self, "_fv_nodes", {}).get(slot)
        if nn is None:
            raise NebError(3, "fastvol_get: empty slot")
        v = np.empty((4, nn))
        self._ck(self._L.neb_fastvol_get(self._h, slot, _ptr(v)))
        return v

    def voxelize_space_charge(self, origin, voxel, dims) -> int:
        """neb_voxelize_space_charge (Alg. 3): the held point charges become line charges; returns their number."""
        origin = np.ascontiguousarray(origin, dtype=np.float64)
        voxel = np.ascontiguousarray(voxel, dtype=np.float64)
        dims = np.ascontiguousarray(dims, dtype=np.int32)
        if origin.shape != (3,) or voxel.shape != (3,) or dims.shape != (3,):
            raise ValueError("origin, voxel and dims must hold 3 values")
        nl = C.c_int64(0)
        self._ck(self._L.neb_voxelize_space_charge(self._h, _ptr(origin), _ptr(voxel), _ptr(dims), C.byref(nl)))
        self._n_lines = int(nl.value)
        return self._n_lines

    def get_line_charges(self):
        """(5, n_lines): x, y, z_start, z_stop, lambda (test hook)."""
        out = np.empty((5, getattr(self, "_n_lines", 0)))
        self._ck(self._L.neb_get_line_charges(self._h, _ptr(out)))
        return out

    def push(self, pos, E, mu_dt: float):
        q = int(pos.shape[1])
        self._ck(self._L.neb_push(self._h, q, _ptr(pos), _ptr(E), float(mu_dt)))
        return pos

    def get_matrix(self):
        K = np.empty((self.n, self.n))
        self._ck(self._L.neb_get_matrix(self._h, _ptr(K)))
        return K.T            # column-major n*n -> K[i, j]

    def get_matrix_rows(self, rows):
        """K[rows, :] (len(rows), n), unscaled, caller's order (test hook; before the first solve)."""
        rows = np.ascontiguousarray(rows, dtype=np.int32)
        out = np.empty((rows.shape[0], self.n))
        self._ck(self._L.neb_get_matrix_rows(self._h, rows.shape[0], _ptr(rows), _ptr(out)))
        return out

    def get_rhs(self):
        b = np.empty(self.n)
        self._ck(self._L.neb_get_rhs(self._h, _ptr(b)))
        return b

    def fp64_peak(self, kind: int) -> float:
        v = C.c_double(0.0)
        self._ck(self._L.neb_fp64_peak(self._h, kind, C.byref(v)))
        return v.value

    def stage_ms(self):
        out = {}
        for s, name in enumerate(STAGES):
            ms, ln = C.c_double(0.0), C.c_int64(0)
            self._ck(self._L.neb_stage_ms(self._h, s, C.byref(ms), C.byref(ln)))
            out[name] = (ms.value, ln.value)
        return out

    def counter(self, which: int) -> float:
        """neb_get_counter: 0 = flop of the DMMA trailing updates, 1 = flop of the whole LU, 2 = matrix bytes written."""
        v = C.c_double(0.0)
        self._ck(self._L.neb_get_counter(self._h, which, C.byref(v)))
        return v.value

    def reset_stats(self):
        self._ck(self._L.neb_reset_stats(self._h))

    def launch_count(self) -> int:
        return int(self._L.neb_launch_count(self._h))

    def set_svd_cutoff(self, rcond: float):
        self._ck(self._L.neb_set_svd_cutoff(self._h, float(rcond)))

    def get_singular_values(self, npad: int):
        """(singular values in column order (npad), sweeps) of the resident SVD factors (test hook)."""
        s, sw = np.empty(npad), C.c_int32(0)
        self._ck(self._L.neb_get_singular_values(self._h, _ptr(s), C.byref(sw)))
        return s, int(sw.value)

    # ---- scale-out of the solve (neb_dist_*): device tensors only; the exchanges are parallel.dist_solve's
    def dist_configure(self, rank: int, world: int):
        self._ck(self._L.neb_dist_configure(self._h, rank, world))

    def dist_npad(self) -> int:
        return int(self._L.neb_dist_npad(self._h))

    def dist_row_scales(self, scales, set_: bool):
        self._ck(self._L.neb_dist_row_scales(self._h, _ptr(scales), 1 if set_ else 0))

    def dist_factor_block(self, g: int, panel, piv, stream=None):
        self._ck(self._L.neb_dist_factor_block(self._h, g, _ptr(panel), _ptr(piv), C.c_void_p(stream.cuda_stream) if stream is not None else None))

    def dist_apply_block(self, g: int, panel, piv, part: int = 0):
        self._ck(self._L.neb_dist_apply_block(self._h, g, _ptr(panel), _ptr(piv), part))

    def dist_finish_factor(self) -> int:
        s = C.c_int32(0)
        self._ck(self._L.neb_dist_finish_factor(self._h, C.byref(s)))
        return int(s.value)

    def dist_rhs(self, y):
        self._ck(self._L.neb_dist_rhs(self._h, _ptr(y)))

    def dist_tri_block(self, upper: bool, g: int, y, acc):
        self._ck(self._L.neb_dist_tri_block(self._h, 1 if upper else 0, g, _ptr(y), _ptr(acc)))

    def dist_set_solution(self, x, out=None):
        self._ck(self._L.neb_dist_set_solution(self._h, _ptr(x), _ptr(out)))
        return out
