"""Seeded synthetic workloads C0..C4 = BASELINE.json configs[0..4] (recipes: SURVEY.md §8(d),
readings S12, S19-S23; restated in DESIGN.md §4).

Input generation only: geometry, boundary values, points and charges.  Nothing here evaluates
a potential, a field or a matrix entry.  All lengths are emitted in metres (SI), SoA layout
(3, n) as the C ABI in include/neb.h wants.

Element convention (include/neb.h): v0 = corner / right-angle vertex / wire start, e1 and e2 the
two perpendicular edge vectors from v0, unit normal n = e2 x e1 / |e2 x e1|.
"""
from dataclasses import dataclass, field
import numpy as np

from . import rng

RECT, TRI, WIRE = 0, 1, 2
DIRICHLET, DIELECTRIC = 0, 1
MM = 1.0e-3
EPS_FR4 = 4.4
Q_E = 1.602176634e-19        # S23
MU_ION = 1.5e-4              # m^2/(V s)  (S23: 1.5 cm^2/(V s))
DT_STEP = 1.0e-9             # s          (S23)


@dataclass
class Problem:
    name: str
    kind: np.ndarray
    v0: np.ndarray
    e1: np.ndarray
    e2: np.ndarray
    radius: np.ndarray
    bc_kind: np.ndarray
    bc_value: np.ndarray
    eps_plus: np.ndarray
    eps_minus: np.ndarray
    img_shift: np.ndarray | None = None          # (3, n_img), includes (0,0,0); None = no copies
    points: np.ndarray | None = None             # (3, m)
    charge_pos: np.ndarray | None = None         # (3, q)
    charge_q: np.ndarray | None = None           # (q,)
    meta: dict = field(default_factory=dict)

    @property
    def n(self) -> int:
        return int(self.kind.shape[0])

    @property
    def n_img(self) -> int:
        return 1 if self.img_shift is None else int(self.img_shift.shape[1])

    def normals(self) -> np.ndarray:
        """(3, n) unit normals by the ABI convention (geometry bookkeeping, not method arithmetic)."""
        c = np.cross(self.e2.T, self.e1.T).T
        return c / np.linalg.norm(c, axis=0)

    def centroids(self) -> np.ndarray:
        """(3, n) default collocation points (reading S4): rectangle centre, triangle v0+(e1+e2)/3,
        wire: mid-length on the surface (offset by radius along a fixed perpendicular)."""
        c = np.where(self.kind == RECT, 0.5, 1.0 / 3.0)[None, :] * (self.e1 + self.e2) + self.v0
        w = self.kind == WIRE
        if np.any(w):
            c[:, w] = self.v0[:, w] + 0.5 * self.e1[:, w] + self.radius[w] * wire_perp(self.e1[:, w])
        return c


def wire_perp(e1: np.ndarray) -> np.ndarray:
    """A unit vector perpendicular to each wire axis: axis x (least-aligned coordinate axis)."""
    t = e1 / np.linalg.norm(e1, axis=0)
    k = np.argmin(np.abs(t), axis=0)
    a = np.zeros_like(t)
    a[k, np.arange(t.shape[1])] = 1.0
    p = np.cross(t.T, a.T).T
    return p / np.linalg.norm(p, axis=0)


class _Builder:
    """Collects elements (in mm) and emits SI SoA arrays."""

    def __init__(self):
        self.kind, self.v0, self.e1, self.e2 = [], [], [], []
        self.bck, self.bcv, self.ep, self.em = [], [], [], []

    def _orient(self, ea, eb, normal):
        ea = np.asarray(ea, float); eb = np.asarray(eb, float)
        if np.dot(np.cross(eb, ea), normal) > 0:
            return ea, eb
        return eb, ea

    def add(self, kind, v0, ea, eb, normal, bc_kind, bc_value, eps_plus=1.0, eps_minus=1.0):
        e1, e2 = self._orient(ea, eb, np.asarray(normal, float))
        self.kind.append(kind); self.v0.append(np.asarray(v0, float)); self.e1.append(e1); self.e2.append(e2)
        self.bck.append(bc_kind); self.bcv.append(bc_value); self.ep.append(eps_plus); self.em.append(eps_minus)

    def rect_cells(self, origin, da, db, ia, ib, normal, **bc):
        """One rectangle per (ia[k], ib[k]) cell of the lattice origin + i*da + j*db."""
        origin = np.asarray(origin, float); da = np.asarray(da, float); db = np.asarray(db, float)
        for i, j in zip(ia, ib):
            self.add(RECT, origin + i * da + j * db, da, db, normal, **bc)

    def finish(self, name, scale=MM, **kw) -> Problem:
        n = len(self.kind)
        f = lambda a: np.ascontiguousarray(np.array(a, dtype=np.float64).reshape(n, 3).T) * scale
        return Problem(
            name=name, kind=np.array(self.kind, dtype=np.int32), v0=f(self.v0), e1=f(self.e1), e2=f(self.e2),
            radius=np.zeros(n), bc_kind=np.array(self.bck, dtype=np.int32),
            bc_value=np.array(self.bcv, dtype=np.float64), eps_plus=np.array(self.ep, dtype=np.float64),
            eps_minus=np.array(self.em, dtype=np.float64), **kw)


def _grid_cells(na, nb, keep=None):
    ia, ib = np.meshgrid(np.arange(na), np.arange(nb), indexing="ij")
    ia, ib = ia.ravel(), ib.ravel()
    if keep is not None:
        m = keep(ia, ib)
        ia, ib = ia[m], ib[m]
    return ia, ib


# ----------------------------------------------------------------------------------------------
# C0: single square plate
# ----------------------------------------------------------------------------------------------
def plate(n_side: int = 16, side_mm: float = 10.0, volt: float = 1.0, m_points: int = 1000, seed: int = 0) -> Problem:
    """C0: plate [-5,5]^2 mm in z=0, n_side x n_side rectangles, 1 V, normal +z; points uniform in
    [-10,10]^3 mm (BASELINE.json configs[0])."""
    b = _Builder()
    p = side_mm / n_side
    ia, ib = _grid_cells(n_side, n_side)
    b.rect_cells((-side_mm / 2, -side_mm / 2, 0.0), (p, 0, 0), (0, p, 0), ia, ib, (0, 0, 1),
                 bc_kind=DIRICHLET, bc_value=volt)
    pts = np.stack([rng.uniform(seed, m_points, -side_mm, side_mm, offset=k * m_points) for k in range(3)]) * MM
    return b.finish(f"C0_plate{n_side}", points=pts, meta=dict(side=side_mm * MM, n_side=n_side, volt=volt))


# ----------------------------------------------------------------------------------------------
# C1: conducting cube
# ----------------------------------------------------------------------------------------------
def cube(n_side: int = 32, side_mm: float = 10.0, volt: float = 1.0, m_points: int = 100_000, seed: int = 1,
         box_mm: float = 30.0) -> Problem:
    """C1: cube [-5,5]^3 mm, 6 faces x n_side^2 rectangles, outward normals, 1 V; points uniform in the
    30 mm cube around it (BASELINE.json configs[1])."""
    b = _Builder()
    h = side_mm / 2
    p = side_mm / n_side
    ia, ib = _grid_cells(n_side, n_side)
    ax = np.eye(3)
    for k in range(3):                      # face normal axis
        a, c = ax[(k + 1) % 3], ax[(k + 2) % 3]
        for s in (+1.0, -1.0):
            origin = s * h * ax[k] - h * a - h * c
            b.rect_cells(origin, p * a, p * c, ia, ib, s * ax[k], bc_kind=DIRICHLET, bc_value=volt)
    pts = np.stack([rng.uniform(seed, m_points, -box_mm / 2, box_mm / 2, offset=k * m_points) for k in range(3)]) * MM
    return b.finish(f"C1_cube{n_side}", points=pts, meta=dict(side=side_mm * MM, n_side=n_side, volt=volt))


# ----------------------------------------------------------------------------------------------
# C2/C3: THGEM-like foils
# ----------------------------------------------------------------------------------------------
def _foil(b: _Builder, d: int, zc: float, xc: float, v_top: float, v_bot: float):
    """One THGEM-like foil (SURVEY §8(d) C2 recipe) centred at height zc (mm), hole centre (xc, 0) mm,
    meshed at pitch 1/d mm inside the cell x,y in [-0.5,0.5] mm (panels wrapped periodically in x)."""
    assert d % 10 == 0
    p = 1.0 / d
    nh, nr, nc = (2 * d) // 10, (3 * d) // 10, d // 2          # half-widths in cells: hole 0.2, rim 0.3, cell 0.5
    zt, zb = 0.25, 0.285                                       # slab half-thickness, copper outer face
    gas = dict(bc_kind=DIELECTRIC, bc_value=0.0, eps_plus=1.0, eps_minus=EPS_FR4)
    n0 = len(b.kind)

    def cheb(i, j):                                            # Chebyshev ring index of cell (i,j) about the hole centre
        ci = np.where(i >= nc, i - nc, nc - 1 - i)
        cj = np.where(j >= nc, j - nc, nc - 1 - j)
        return np.maximum(ci, cj)

    org = (xc - 0.5, -0.5)
    for sgn, volt in ((+1.0, v_top), (-1.0, v_bot)):
        cu = dict(bc_kind=DIRICHLET, bc_value=volt)
        # copper outer face and copper/slab contact face (S9: conductor panels only)
        ia, ib = _grid_cells(d, d, lambda i, j: cheb(i, j) >= nr)
        b.rect_cells((org[0], org[1], zc + sgn * zb), (p, 0, 0), (0, p, 0), ia, ib, (0, 0, sgn), **cu)
        b.rect_cells((org[0], org[1], zc + sgn * zt), (p, 0, 0), (0, p, 0), ia, ib, (0, 0, -sgn), **cu)
        # copper rim walls at |x-xc| = 0.3 or |y| = 0.3, 2 strips over 35 um, normal toward the hole axis
        hz = (zb - zt) / 2
        z_lo = zc + (zt if sgn > 0 else -zb)
        ia, ib = _grid_cells(2 * nr, 2)
        for s in (+1.0, -1.0):
            b.rect_cells((xc - nr * p, s * nr * p, z_lo), (p, 0, 0), (0, 0, hz), ia, ib, (0, -s, 0), **cu)
            b.rect_cells((xc + s * nr * p, -nr * p, z_lo), (0, p, 0), (0, 0, hz), ia, ib, (-s, 0, 0), **cu)
        # exposed slab rim (dielectric rows, n from slab into gas); corner blocks split into right triangles
        z = zc + sgn * zt
        ia, ib = _grid_cells(d, d, lambda i, j: (cheb(i, j) >= nh) & (cheb(i, j) < nr))
        for i, j in zip(ia, ib):
            x0, y0 = org[0] + i * p, org[1] + j * p
            ci = i - nc if i >= nc else nc - 1 - i
            cj = j - nc if j >= nc else nc - 1 - j
            if ci >= nh and cj >= nh:                          # corner block: diagonal points at the hole
                if (i >= nc) == (j >= nc):                     # diagonal (x0,y0)-(x0+p,y0+p)
                    b.add(TRI, (x0 + p, y0, z), (-p, 0, 0), (0, p, 0), (0, 0, sgn), **gas)
                    b.add(TRI, (x0, y0 + p, z), (p, 0, 0), (0, -p, 0), (0, 0, sgn), **gas)
                else:                                          # diagonal (x0+p,y0)-(x0,y0+p)
                    b.add(TRI, (x0, y0, z), (p, 0, 0), (0, p, 0), (0, 0, sgn), **gas)
                    b.add(TRI, (x0 + p, y0 + p, z), (-p, 0, 0), (0, -p, 0), (0, 0, sgn), **gas)
            else:
                b.add(RECT, (x0, y0, z), (p, 0, 0), (0, p, 0), (0, 0, sgn), **gas)
    # hole walls |x-xc| = 0.2 or |y| = 0.2 through the slab, n into the hole (slab -> gas)
    ia, ib = _grid_cells(2 * nh, nc)                            # 0.4 mm along, 0.5 mm in z
    for s in (+1.0, -1.0):
        b.rect_cells((xc - nh * p, s * nh * p, zc - zt), (p, 0, 0), (0, 0, p), ia, ib, (0, -s, 0), **gas)
        b.rect_cells((xc + s * nh * p, -nh * p, zc - zt), (0, p, 0), (0, 0, p), ia, ib, (-s, 0, 0), **gas)
    # periodic wrap in x: panels whose centre lies beyond +0.5 mm move by one pitch
    for k in range(n0, len(b.kind)):
        w = 0.5 if b.kind[k] == RECT else 1.0 / 3.0
        cx = b.v0[k][0] + w * (b.e1[k][0] + b.e2[k][0])
        if cx > 0.5:
            b.v0[k] = b.v0[k] - np.array([1.0, 0.0, 0.0])


def _planes(b: _Builder, n_plane: int, v_drift=-2000.0, v_ind=0.0):
    p = 1.0 / n_plane
    ia, ib = _grid_cells(n_plane, n_plane)
    b.rect_cells((-0.5, -0.5, 3.0), (p, 0, 0), (0, p, 0), ia, ib, (0, 0, -1), bc_kind=DIRICHLET, bc_value=v_drift)
    b.rect_cells((-0.5, -0.5, -2.0), (p, 0, 0), (0, p, 0), ia, ib, (0, 0, 1), bc_kind=DIRICHLET, bc_value=v_ind)


def _grid_points(n: int) -> np.ndarray:
    """n^3 cell-centred nodes spanning x,y in [-0.5,0.5] mm, z in [-2,3] mm; x fastest."""
    g = (np.arange(n) + 0.5) / n
    x, y, z = -0.5 + g, -0.5 + g, -2.0 + 5.0 * g
    zz, yy, xx = np.meshgrid(z, y, x, indexing="ij")
    return np.stack([xx.ravel(), yy.ravel(), zz.ravel()]) * MM


def image_shifts(k: int = 2, pitch_mm: float = 1.0) -> np.ndarray:
    """(3, (2k+1)^2) periodic copies in x,y (reading S12); shift (0,0,0) first."""
    r = np.arange(-k, k + 1)
    mx, my = np.meshgrid(r, r, indexing="ij")
    s = np.stack([mx.ravel(), my.ravel(), np.zeros(mx.size)]).astype(np.float64) * pitch_mm * MM
    order = np.argsort(np.abs(s[0]) + np.abs(s[1]), kind="stable")
    return np.ascontiguousarray(s[:, order])


def thgem(d: int = 60, n_plane: int = 50, n_grid: int = 100) -> Problem:
    """C2: one THGEM-like cell (BASELINE.json configs[2]); d = pitch divisor (cells per mm)."""
    b = _Builder()
    _foil(b, d, 0.0, 0.0, 0.0, -1000.0)                         # S19
    _planes(b, n_plane)
    return b.finish(f"C2_thgem{d}", points=_grid_points(n_grid), meta=dict(d=d, n_plane=n_plane))


def double_thgem(d: int = 70, n_plane: int = 74, m_points: int = 10_000_000, seed: int = 3, k_img: int = 2) -> Problem:
    """C3: two staggered foils + 5x5 image copies (BASELINE.json configs[3]; S20, S21, S12)."""
    b = _Builder()
    _foil(b, d, 0.0, 0.0, 0.0, -1000.0)
    _foil(b, d, 2.0, 0.5, -1000.0, -2000.0)
    _planes(b, n_plane)
    lo, hi = (-0.5, -0.5, -2.0), (0.5, 0.5, 3.0)
    pts = np.stack([rng.uniform(seed, m_points, lo[k], hi[k], offset=k * m_points) for k in range(3)]) * MM
    return b.finish(f"C3_double_thgem{d}", points=pts, img_shift=image_shifts(k_img) if k_img > 0 else None,
                    meta=dict(d=d, n_plane=n_plane))


def space_charge(base: Problem, q_count: int = 1_000_000, sigma_mm: float = 0.1, seed: int = 4) -> Problem:
    """C4: q_count charges of +1e, centres Gaussian(sigma) per axis about the stage-1 hole centre (S22, S23)."""
    pos = np.stack([rng.normal(seed, q_count, offset=2 * k * q_count) for k in range(3)]) * (sigma_mm * MM)
    base.charge_pos = np.ascontiguousarray(pos)
    base.charge_q = np.full(q_count, Q_E)
    base.name = base.name + f"+sc{q_count}"
    base.meta.update(mu=MU_ION, dt=DT_STEP, steps=10)
    return base


# ----------------------------------------------------------------------------------------------
# small mixed-kind problems for unit/parity tests
# ----------------------------------------------------------------------------------------------
def random_elements(n: int, seed: int, kinds=(RECT, TRI, WIRE), size_mm=(0.05, 1.0), box_mm: float = 2.0,
                    m_points: int = 0, dielectric_fraction: float = 0.0) -> Problem:
    """n randomly placed, randomly oriented elements of mixed kinds inside a box (tests only)."""
    u = lambda k, lo, hi: rng.uniform(seed, n, lo, hi, offset=k * n)
    kind = np.array(kinds, dtype=np.int32)[(u(0, 0, 1) * len(kinds)).astype(int) % len(kinds)]
    v0 = np.stack([u(1, -box_mm, box_mm), u(2, -box_mm, box_mm), u(3, -box_mm, box_mm)])
    a = np.stack([rng.normal(seed + 1000, n, offset=k * 2 * n) for k in range(3)])
    c = np.stack([rng.normal(seed + 2000, n, offset=k * 2 * n) for k in range(3)])
    a /= np.linalg.norm(a, axis=0)
    c -= a * np.sum(a * c, axis=0)
    c /= np.linalg.norm(c, axis=0)
    e1 = a * u(20, *size_mm)
    e2 = c * u(21, *size_mm)
    radius = np.where(kind == WIRE, u(22, 0.005, 0.02), 0.0)
    diel = (u(23, 0, 1) < dielectric_fraction) & (kind != WIRE)
    pr = Problem(
        name=f"random{n}_s{seed}", kind=kind, v0=v0 * MM, e1=e1 * MM, e2=e2 * MM, radius=radius * MM,
        bc_kind=np.where(diel, DIELECTRIC, DIRICHLET).astype(np.int32),
        bc_value=np.where(diel, 0.0, u(24, -100.0, 100.0)),
        eps_plus=np.ones(n), eps_minus=np.where(diel, u(25, 2.0, 10.0), 1.0))
    if m_points:
        pr.points = np.stack([rng.uniform(seed + 1, m_points, -1.5 * box_mm, 1.5 * box_mm, offset=k * m_points)
                              for k in range(3)]) * MM
    return pr


def with_coincident_panels(pr: Problem, idx) -> Problem:
    """pr with the elements idx listed a second time (appended): coincident panels, the "overlapping surfaces" that the
    repetition of primitives produces and that make the influence matrix exactly rank-deficient (OptSVD tests)."""
    idx = np.asarray(idx, dtype=np.int64)
    cat1 = lambda a: np.concatenate([a, a[idx]])
    cat3 = lambda a: np.ascontiguousarray(np.concatenate([a, a[:, idx]], axis=1))
    return Problem(name=pr.name + "_overlap", kind=cat1(pr.kind), v0=cat3(pr.v0), e1=cat3(pr.e1), e2=cat3(pr.e2),
                   radius=cat1(pr.radius), bc_kind=cat1(pr.bc_kind), bc_value=cat1(pr.bc_value), eps_plus=cat1(pr.eps_plus),
                   eps_minus=cat1(pr.eps_minus), img_shift=pr.img_shift, points=pr.points, meta=dict(pr.meta, duplicated=idx))


def by_name(name: str) -> Problem:
    """Full-size BASELINE configs by short name."""
    if name == "C0":
        return plate()
    if name == "C1":
        return cube()
    if name == "C2":
        return thgem()
    if name == "C3":
        return double_thgem()
    if name == "C4":
        return space_charge(double_thgem(m_points=0))
    raise KeyError(name)
