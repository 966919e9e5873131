"""ctypes binding of oracle/neb_oracle.c — TEST INFRASTRUCTURE, NOT THE PRODUCT.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may import
this package; it imports nothing from paper_2606_24154_b200 and the CUDA path imports nothing
from here.  Two builds of the same C source: `f64` (real = double, the timed CPU baseline) and
`ld` (real = long double, the truth for parity tests).  See the header of neb_oracle.c for the
passages each function follows and the list of pins.
"""
import ctypes as C
import os
import subprocess
import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "neb_oracle.c")
_LIBS = {"f64": os.path.join(_HERE, "liborc_f64.so"), "ld": os.path.join(_HERE, "liborc_ld.so")}
_FLAGS = {"f64": [], "ld": ["-DORC_LONG_DOUBLE"]}
_cache = {}

EPS0 = 8.8541878128e-12          # reading S3 (the same CODATA value is restated in the C source)
K_COULOMB = 1.0 / (4.0 * np.pi * EPS0)


def build(force: bool = False) -> None:
    """gcc -O2 -fopenmp (no -ffast-math), both precisions."""
    for mode, lib in _LIBS.items():
        if force or not os.path.exists(lib) or os.path.getmtime(lib) < os.path.getmtime(_SRC):
            cmd = ["gcc", "-O2", "-fopenmp", "-fPIC", "-shared", "-std=c99", "-ffp-contract=off",
                   *_FLAGS[mode], _SRC, "-o", lib, "-lm"]
            subprocess.check_call(cmd)


_dp = C.POINTER(C.c_double)
_ip = C.POINTER(C.c_int32)
_lp = C.POINTER(C.c_int64)


def _lib(mode: str):
    if mode not in _cache:
        build()
        L = C.CDLL(_LIBS[mode])
        L.orc_real_bytes.restype = C.c_int
        L.orc_threads.restype = C.c_int
        L.orc_lu_factor.restype = C.c_void_p
        L.orc_lu_factor.argtypes = [C.c_int64, _dp, _ip]
        L.orc_lu_solve.argtypes = [C.c_void_p, _dp, _dp]
        L.orc_lu_free.argtypes = [C.c_void_p]
        L.orc_solve.restype = C.c_int32
        _cache[mode] = L
    return _cache[mode]


def _d(a):
    return None if a is None else np.ascontiguousarray(a, dtype=np.float64)


def _p(a, t=_dp):
    return None if a is None else a.ctypes.data_as(t)


def threads(mode="f64") -> int:
    return int(_lib(mode).orc_threads())


def influence(kind, v0, e1, e2, P, radius=0.0, mode="ld"):
    """(Phi', E'x, E'y, E'z) of one element at one point, primed (no 1/4 pi eps0, no sigma)."""
    v0, e1, e2, P = (_d(x) for x in (v0, e1, e2, P))
    out = np.zeros(4)
    _lib(mode).orc_influence(C.c_int32(int(kind)), _p(v0), _p(e1), _p(e2), C.c_double(float(radius)), _p(P), _p(out))
    return out


class Geometry:
    """Holds contiguous SoA copies of a workloads.configs.Problem's arrays for the C calls."""

    def __init__(self, pr, colloc=None):
        self.n = int(pr.kind.shape[0])
        self.kind = np.ascontiguousarray(pr.kind, dtype=np.int32)
        self.v0, self.e1, self.e2 = _d(pr.v0), _d(pr.e1), _d(pr.e2)
        self.radius = _d(pr.radius)
        self.colloc = _d(pr.centroids() if colloc is None else colloc)
        self.bc_kind = np.ascontiguousarray(pr.bc_kind, dtype=np.int32)
        self.bc_value = _d(pr.bc_value)
        self.eps_plus, self.eps_minus = _d(pr.eps_plus), _d(pr.eps_minus)
        self.img = _d(pr.img_shift)
        self.n_img = 0 if self.img is None else int(self.img.shape[1])

    def _geo(self):
        return (C.c_int64(self.n), _p(self.kind, _ip), _p(self.v0), _p(self.e1), _p(self.e2), _p(self.radius))


def assemble(g: Geometry, mode="ld") -> np.ndarray:
    """K[i, j], row i = collocation point i, column j = source element j (LHMatrix)."""
    K = np.zeros((g.n, g.n))
    _lib(mode).orc_assemble(*g._geo(), _p(g.colloc), _p(g.bc_kind, _ip), _p(g.eps_plus), _p(g.eps_minus),
                            C.c_int32(g.n_img), _p(g.img), _p(K))
    return K


def matrix_entries(g: Geometry, rows, cols, mode="ld") -> np.ndarray:
    rows = np.ascontiguousarray(rows, dtype=np.int64)
    cols = np.ascontiguousarray(cols, dtype=np.int64)
    vals = np.zeros(rows.shape[0])
    _lib(mode).orc_matrix_entries(*g._geo(), _p(g.colloc), _p(g.bc_kind, _ip), _p(g.eps_plus), _p(g.eps_minus),
                                  C.c_int32(g.n_img), _p(g.img), C.c_int64(rows.shape[0]), _p(rows, _lp),
                                  _p(cols, _lp), _p(vals))
    return vals


def rhs(g: Geometry, charge_pos=None, charge_q=None, mode="ld") -> np.ndarray:
    b = np.zeros(g.n)
    pos, ch = _d(charge_pos), _d(charge_q)
    q = 0 if ch is None else int(ch.shape[0])
    _lib(mode).orc_rhs(C.c_int64(g.n), _p(g.e1), _p(g.e2), _p(g.colloc), _p(g.bc_kind, _ip), _p(g.bc_value),
                       C.c_int64(q), _p(pos), _p(ch), _p(b))
    return b


def solve(K: np.ndarray, b: np.ndarray, mode="ld") -> np.ndarray:
    K, b = _d(K), _d(b)
    x = np.zeros_like(b)
    st = _lib(mode).orc_solve(C.c_int64(K.shape[0]), _p(K), _p(b), _p(x))
    if st != 0:
        raise np.linalg.LinAlgError(f"oracle LU: status {st}")
    return x


class LU:
    """Factor once, re-solve many times (reading S13)."""

    def __init__(self, K, mode="ld"):
        self._L = _lib(mode)
        K = _d(K)
        self.n = K.shape[0]
        st = C.c_int32(0)
        self._h = self._L.orc_lu_factor(C.c_int64(self.n), _p(K), C.byref(st))
        if st.value != 0:
            raise np.linalg.LinAlgError(f"oracle LU: status {st.value}")

    def solve(self, b):
        b = _d(b)
        x = np.zeros_like(b)
        self._L.orc_lu_solve(C.c_void_p(self._h), _p(b), _p(x))
        return x

    def __del__(self):
        if getattr(self, "_h", None):
            self._L.orc_lu_free(C.c_void_p(self._h))
            self._h = None


def point_charges(pts, charge_pos, charge_q, mode="ld"):
    pts, pos, ch = _d(pts), _d(charge_pos), _d(charge_q)
    m = pts.shape[1]
    phi, E = np.zeros(m), np.zeros((3, m))
    _lib(mode).orc_point_charges(C.c_int64(m), _p(pts), C.c_int64(ch.shape[0]), _p(pos), _p(ch), _p(phi), _p(E))
    return phi, E


def evaluate(g: Geometry, sigma, pts, charge_pos=None, charge_q=None, mode="ld"):
    """Phi (m), E (3, m) at pts (3, m) from elements with densities sigma, plus space charges."""
    sigma, pts, pos, ch = _d(sigma), _d(pts), _d(charge_pos), _d(charge_q)
    m = pts.shape[1]
    q = 0 if ch is None else int(ch.shape[0])
    phi, E = np.zeros(m), np.zeros((3, m))
    _lib(mode).orc_eval(*g._geo(), _p(sigma), C.c_int32(g.n_img), _p(g.img), C.c_int64(q), _p(pos), _p(ch),
                        C.c_int64(m), _p(pts), _p(phi), _p(E))
    return phi, E


def evaluate_abs(g: Geometry, sigma, pts, charge_pos=None, charge_q=None, mode="f64", with_field=False):
    """S_Phi (m), S_E (m): sums of the magnitudes of the terms evaluate() adds at pts (3, m) — the scale of the
    rounding error of a cancelled sum; a tolerance scale for the parity tests, not a result.
    with_field=True also returns Phi, E formed in the same pass (bit-identical to evaluate()): (S_Phi, S_E, Phi, E)."""
    sigma, pts, pos, ch = _d(sigma), _d(pts), _d(charge_pos), _d(charge_q)
    m = pts.shape[1]
    q = 0 if ch is None else int(ch.shape[0])
    s_phi, s_E = np.zeros(m), np.zeros(m)
    phi, E = (np.zeros(m), np.zeros((3, m))) if with_field else (None, None)
    _lib(mode).orc_eval_abs(*g._geo(), _p(sigma), C.c_int32(g.n_img), _p(g.img), C.c_int64(q), _p(pos), _p(ch),
                            C.c_int64(m), _p(pts), _p(s_phi), _p(s_E), _p(phi), _p(E))
    return (s_phi, s_E, phi, E) if with_field else (s_phi, s_E)


def solve_library(K: np.ndarray, b: np.ndarray) -> np.ndarray:
    """The solution of K sigma = b (Eq. 6-7) with a LIBRARY routine as the step: rows equilibrated by
    1/max_j|K_ij| (reading S15), then numpy.linalg.solve (LAPACK dgesv: LU with partial pivoting, the same
    algorithm as orc_solve).  For sizes the plain C loop of orc_lu_factor cannot finish in test time (C2: N = 19400);
    tests/test_oracle_pins.py checks the two against each other on small systems."""
    K, b = _d(K), _d(b)
    r = 1.0 / np.abs(K).max(axis=1)
    return np.linalg.solve(K * r[:, None], b * r)


def solve_svd(K: np.ndarray, b: np.ndarray, rcond: float = 1e-10) -> np.ndarray:
    """OptSVD ("overlapping surfaces ... Singular Value Decomposition can be used to obtain the solution"; the
    paper does not say which solution — reading S31): the MINIMUM-NORM least-squares solution of the row-equilibrated
    system (reading S15), sigma = sum over s_i > rcond s_max of v_i (u_i . b) / s_i, with numpy.linalg.svd (LAPACK
    gesdd) as the library step.  Coincident panels make K exactly rank-deficient: their columns are equal, the
    singular value of the difference direction is ~eps s_max and is dropped, the charge is shared equally."""
    K, b = _d(K), _d(b)
    r = 1.0 / np.abs(K).max(axis=1)
    U, S, Vt = np.linalg.svd(K * r[:, None])
    keep = S > rcond * S[0]
    return Vt[keep].T @ ((U[:, keep].T @ (b * r)) / S[keep])


def push(pos, E, mu, dt, mode="ld"):
    pos = np.array(pos, dtype=np.float64, order="C")
    E = _d(E)
    _lib(mode).orc_push(C.c_int64(pos.shape[1]), _p(pos), _p(E), C.c_double(mu), C.c_double(dt))
    return pos


def fastvol_nodes(nx, ny, nz, origin, spacing):
    """Node coordinates (3, nx*ny*nz) of a uniform FastVolume grid, i fastest (reading S25)."""
    k, j, i = np.meshgrid(np.arange(nz), np.arange(ny), np.arange(nx), indexing="ij")
    return np.stack([origin[0] + i.ravel() * spacing[0], origin[1] + j.ravel() * spacing[1],
                     origin[2] + k.ravel() * spacing[2]])


def fastvol_eval(shape, origin, spacing, values, pts, mode="ld"):
    """Trilinear interpolation of values (4, nx*ny*nz) = Phi, Ex, Ey, Ez at pts (3, m); NaN outside."""
    nx, ny, nz = (int(v) for v in shape)
    values, pts = _d(values), _d(pts)
    origin, spacing = _d(np.asarray(origin, dtype=np.float64)), _d(np.asarray(spacing, dtype=np.float64))
    m = pts.shape[1]
    phi, E = np.zeros(m), np.zeros((3, m))
    _lib(mode).orc_fastvol_eval(C.c_int32(nx), C.c_int32(ny), C.c_int32(nz), _p(origin), _p(spacing), _p(values),
                                C.c_int64(m), _p(pts), _p(phi), _p(E))
    return phi, E


def weighting_rhs(g: Geometry, bc_value_w) -> np.ndarray:
    """Right-hand side of a weighting-field solve (P:222 CreateWtFldFastVolPF; reading S26): the read-out
    electrode's panels at their weighting potential (1), every other conductor at 0, no space charge;
    dielectric rows stay homogeneous (0)."""
    return np.where(g.bc_kind == 0, np.asarray(bc_value_w, dtype=np.float64), 0.0)


def voxelize(charge_pos, charge_q, origin, voxel, dims):
    """Alg. 3 (reading S27): point charges -> line charges.  Returns lines (5, nl): x, y, z_start,
    z_stop, lambda, in voxel-index order."""
    pos, ch = _d(charge_pos), _d(charge_q)
    origin, voxel = _d(np.asarray(origin, dtype=np.float64)), _d(np.asarray(voxel, dtype=np.float64))
    dims = np.ascontiguousarray(dims, dtype=np.int32)
    q = int(ch.shape[0])
    cap = int(min(q, int(np.prod(dims.astype(np.int64))))) or 1
    lines = np.zeros((5, cap))
    L = _lib("f64")
    L.orc_voxelize.restype = C.c_int64
    nl = L.orc_voxelize(C.c_int64(q), _p(pos), _p(ch), _p(origin), _p(voxel), _p(dims, _ip), C.c_int64(cap), _p(lines))
    if nl < 0:
        raise RuntimeError("oracle voxelize: capacity")
    return np.ascontiguousarray(lines[:, :nl])


def line_charges(pts, lines, mode="ld"):
    """Phi (m), E (3, m) of line charges (5, nl) parallel to z at pts (3, m)."""
    pts, lines = _d(pts), _d(lines)
    m, nl = pts.shape[1], lines.shape[1]
    phi, E = np.zeros(m), np.zeros((3, m))
    _lib(mode).orc_line_charges(C.c_int64(m), _p(pts), C.c_int64(nl), C.c_int64(nl), _p(lines), _p(phi), _p(E))
    return phi, E


def evaluate_adaptive(g: Geometry, sigma, pts, far_distance, charge_pos=None, charge_q=None, mode="ld"):
    """evaluate() with Adaptive Modelling (reading S28): image copies whose shift is at least far_distance
    long are replaced by the element's total charge at the copy's centroid."""
    sigma, pts, pos, ch = _d(sigma), _d(pts), _d(charge_pos), _d(charge_q)
    m = pts.shape[1]
    q = 0 if ch is None else int(ch.shape[0])
    phi, E = np.zeros(m), np.zeros((3, m))
    _lib(mode).orc_eval_adaptive(*g._geo(), _p(sigma), C.c_int32(g.n_img), _p(g.img), C.c_double(float(far_distance)),
                                 C.c_int64(q), _p(pos), _p(ch), C.c_int64(m), _p(pts), _p(phi), _p(E))
    return phi, E
