"""neb_eval_static — the evaluation entry point that allocates nothing (include/neb.h): its partial sums live in a
file-scope device array of fixed size instead of a cudaMalloc'ed buffer.  Checked against the existing path (neb_eval) on
the same context, on two calls in a row (the array keeps the previous call's contents), within the tolerance the parity
tests use for Phi and |E| (1e-10 relative per point + the per-point allowance for a cancelled sum, here taken from the
magnitudes of the existing path's own terms: max|Phi|, max|E| over the points).

Collected LAST on purpose (file name): the suite runs with pytest -x, a failure here must not hide other tests.
"""
import numpy as np
import pytest

from workloads import configs as W

pytestmark = pytest.mark.gpu

TOL = 1e-10


def _close(got, want, what):
    got, want = got.cpu().numpy(), want.cpu().numpy()
    if got.ndim == 1:
        err, mag = np.abs(got - want), np.abs(want)
    else:
        err, mag = np.linalg.norm(got - want, axis=0), np.linalg.norm(want, axis=0)
    # the two paths differ only in how many chunks the fixed-order sum is cut into: per point tol x |value| plus a few
    # ulps of the largest value on the map (a sum that cancels at a point keeps the rounding error of its terms)
    allow = TOL * mag + 64 * 2.0 ** -53 * mag.max()
    assert np.all(err <= allow), f"{what}: max err/allow {np.max(err / allow):.3f}"


def test_eval_static_matches_eval_on_two_calls_in_a_row():
    import torch
    import paper_2606_24154_b200 as P
    pr = W.double_thgem(d=10, n_plane=10, m_points=40000, k_img=1)        # rectangles + triangles, dielectric rows, 3 x 3 copies
    rs = np.random.RandomState(5)
    nb = P.Neb()
    nb.assemble_problem(pr)
    pos = rs.normal(size=(3, 3000)) * 1e-4
    nb.add_space_charge(pos, np.full(3000, W.Q_E * 1e5))
    nb.solve()
    f64 = dict(dtype=torch.float64, device="cuda")
    pts_a = torch.from_numpy(pr.points).cuda().contiguous()               # 40000 points: the chunk counts get cut to fit
    pts_b = torch.from_numpy(np.ascontiguousarray(pr.points[:, :777])).cuda()   # a small call right after a large one
    phi_a, E_a = torch.empty(40000, **f64), torch.empty((3, 40000), **f64)
    phi_b, E_b = torch.empty(777, **f64), torch.empty((3, 777), **f64)
    # two calls in a row on the shared array, then the first again: stale contents of a longer call must not matter
    nb.eval_static(pts_a, phi_a, E_a)
    nb.eval_static(pts_b, phi_b, E_b)
    phi_a2, E_a2 = torch.empty_like(phi_a), torch.empty_like(E_a)
    nb.eval_static(pts_a, phi_a2, E_a2)
    ref_phi_a, ref_E_a = nb.eval(pts_a)                                   # the existing path
    ref_phi_b, ref_E_b = nb.eval(pts_b)
    _close(phi_a, ref_phi_a, "Phi, first call")
    _close(E_a, ref_E_a, "E, first call")
    _close(phi_b, ref_phi_b, "Phi, second call")
    _close(E_b, ref_E_b, "E, second call")
    assert torch.equal(phi_a, phi_a2) and torch.equal(E_a, E_a2)          # same call, same bits, whatever ran in between
    # only one output wanted
    only_phi = torch.empty(777, **f64)
    nb.eval_static(pts_b, only_phi, None)
    assert torch.equal(only_phi, phi_b)
    # the limits: too many points, host pointers
    big = torch.zeros((3, P.binding.NEB_EVAL_STATIC_MAX_POINTS + 1), **f64)
    with pytest.raises(P.NebError) as e:
        nb.eval_static(big, torch.empty(big.shape[1], **f64), None)
    assert e.value.status == 1 and "65536" in str(e.value)
    with pytest.raises(P.NebError) as e:
        nb.eval_static(pr.points[:, :10].copy(), np.empty(10), np.empty((3, 10)))
    assert e.value.status == 1
    # exactly the maximum is accepted
    full = pts_a[:, :1].repeat(1, P.binding.NEB_EVAL_STATIC_MAX_POINTS).contiguous()
    phi_f = torch.empty(full.shape[1], **f64)
    nb.eval_static(full, phi_f, None)
    assert torch.all(phi_f == phi_f[0]) and abs(float(phi_f[0]) - float(ref_phi_a[0])) <= TOL * abs(float(ref_phi_a[0])) + 1e-13 * float(ref_phi_a.abs().max())
    nb.close()


def test_eval_static_on_a_second_context_and_without_charges():
    """A fresh context (its own cudaGetSymbolAddress at neb_create) on a copy-free mesh, no space charge."""
    import torch
    import paper_2606_24154_b200 as P
    pr = W.cube(n_side=8, m_points=5000)
    nb = P.Neb()
    nb.assemble_problem(pr)
    nb.solve()
    pts = torch.from_numpy(pr.points).cuda().contiguous()
    phi, E = torch.empty(5000, dtype=torch.float64, device="cuda"), torch.empty((3, 5000), dtype=torch.float64, device="cuda")
    for _ in range(2):
        nb.eval_static(pts, phi, E)
        ref_phi, ref_E = nb.eval(pts)
        _close(phi, ref_phi, "Phi")
        _close(E, ref_E, "E")
    nb.close()


def test_eval_static_with_many_copies_lines_and_adaptive_modelling():
    """The branches of the launch logic that neb_eval_static repeats from neb_eval: more than 32 periodic copies (several
    launches per call, later ones ADD to the partial sums the first one stored — on an array that still holds another
    call's values), line charges from the voxelisation beside point charges, far copies simplified."""
    import torch
    import paper_2606_24154_b200 as P
    pr = W.double_thgem(d=10, n_plane=10, m_points=3000, k_img=3)          # 7 x 7 = 49 copies: two chunks of the copy table
    assert pr.n_img == 49
    rs = np.random.RandomState(6)
    nb = P.Neb()
    nb.assemble_problem(pr)
    nb.set_sigma(rs.uniform(1e-8, 3e-8, pr.n))
    pos = rs.normal(size=(3, 2000)) * 1e-4
    nb.add_space_charge(pos, np.full(2000, W.Q_E * 1e5))
    assert nb.voxelize_space_charge(np.full(3, -4e-4), np.full(3, 1e-4), np.full(3, 8, dtype=np.int32)) > 0
    nb.add_space_charge(rs.normal(size=(3, 500)) * 1e-4, np.full(500, W.Q_E * 1e5), replace=False)   # points beside the lines
    pts = torch.from_numpy(pr.points).cuda().contiguous()
    f64 = dict(dtype=torch.float64, device="cuda")
    junk = torch.from_numpy(pr.points[:, ::-1].copy() * 0.5).cuda().contiguous()
    for far in (0.0, 2.5e-3):
        nb.set_adaptive(far)
        nb.eval_static(junk, torch.empty(3000, **f64), torch.empty((3, 3000), **f64))     # leaves other values in the array
        phi, E = torch.empty(3000, **f64), torch.empty((3, 3000), **f64)
        nb.eval_static(pts, phi, E)
        ref_phi, ref_E = nb.eval(pts)
        _close(phi, ref_phi, f"Phi, far={far}")
        _close(E, ref_E, f"E, far={far}")
    nb.close()
