"""CPU-only checks: the C-ABI library builds in-tree, loads and exports every symbol include/neb.h declares
(no compute call without a GPU); the product path fails loudly without a device; the seeded workload
generators produce the shapes DESIGN.md §4 states."""
import os

import numpy as np
import pytest
import torch

from workloads import configs as W
from workloads import rng


def test_library_exports_every_declared_symbol():
    import paper_2606_24154_b200 as P
    L = P.lib()
    names = P.exported_symbols()
    assert {"neb_create", "neb_destroy", "neb_assemble", "neb_solve", "neb_eval", "neb_add_space_charge",
            "neb_set_sigma", "neb_push", "neb_get_matrix", "neb_get_rhs", "neb_last_error", "neb_set_option",
            "neb_fp64_peak", "neb_stage_ms", "neb_reset_stats", "neb_launch_count"} <= set(names)
    for n in names:
        assert getattr(L, n) is not None
    assert os.path.dirname(P.lib_path()) == os.path.dirname(P.__file__)          # in-tree, not site-packages


@pytest.mark.skipif(torch.cuda.is_available(), reason="only meaningful on a box without a GPU")
def test_no_cpu_fallback():
    import paper_2606_24154_b200 as P
    with pytest.raises(P.NebError):
        P.Neb()
    # the package never imports the oracle
    import sys
    assert "oracle" not in {m.split(".")[0] for m in sys.modules if m.startswith("paper_2606_24154_b200")}
    src_dir = os.path.dirname(P.__file__)
    for root, _, files in os.walk(src_dir):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                text = open(os.path.join(root, f)).read()
                assert "import oracle" not in text and "from oracle" not in text and "neb_oracle" not in text


def test_splitmix64_test_vector_and_stream_slicing():
    # published SplitMix64 outputs for state 0
    assert [int(x) for x in rng.u64(0, 3)] == [0xE220A8397B1DCDAF, 0x6E789E6AA1B965F4, 0x06C45D188009454F]
    a, b = rng.uniform01(7, 10), rng.uniform01(7, 4, offset=6)
    assert np.array_equal(a[6:], b) and np.all((a >= 0) & (a < 1))
    g = rng.normal(3, 200000)
    assert abs(g.mean()) < 0.01 and abs(g.std() - 1) < 0.01


def test_config_shapes():
    c0, c1 = W.plate(), W.cube()
    assert c0.n == 256 and c0.points.shape == (3, 1000) and np.all(np.abs(c0.points) <= 0.01)
    assert c1.n == 6144 and c1.points.shape == (3, 100000) and np.all(np.abs(c1.points) <= 0.015)
    nrm, cen = c1.normals(), c1.centroids()
    assert np.all(np.sum(nrm * cen, axis=0) > 0)                                  # outward normals
    assert np.allclose(np.abs(cen).max(axis=0), 0.005)
    c2 = W.thgem()
    assert c2.n == 19400 and np.sum(c2.kind == W.TRI) == 576 and np.sum(c2.bc_kind == W.DIELECTRIC) == 4608
    assert c2.points.shape == (3, 1000000)
    assert set(np.unique(c2.bc_value[c2.bc_kind == W.DIRICHLET])) == {-2000.0, -1000.0, 0.0}
    area = np.linalg.norm(np.cross(c2.e1.T, c2.e2.T), axis=1) * np.where(c2.kind == W.TRI, 0.5, 1.0)
    # exposed slab rims: 2 x (0.6^2 - 0.4^2) mm^2, hole walls 4 x 0.4 x 0.5 mm^2
    assert abs(area[c2.bc_kind == W.DIELECTRIC].sum() - (2 * 0.2 + 0.8) * 1e-6) < 1e-15
    # dielectric normals point from the slab into the gas: away from the slab's mid-plane or into the hole
    d = c2.bc_kind == W.DIELECTRIC
    n2, p2 = c2.normals()[:, d], c2.centroids()[:, d]
    flat = np.abs(n2[2]) > 0.5
    assert np.all(n2[2, flat] * p2[2, flat] > 0)
    assert np.all(np.sum(n2[:2, ~flat] * p2[:2, ~flat], axis=0) < 0)
    c3 = W.double_thgem(m_points=10)
    assert c3.n == 49928 and c3.n_img == 25 and np.all(c3.img_shift[:, 0] == 0)
    assert np.abs(c3.centroids()[0]).max() < 0.5e-3                               # stage 2 wrapped into the cell
    c4 = W.space_charge(W.plate(), q_count=1000)
    assert c4.charge_pos.shape == (3, 1000) and np.all(c4.charge_q == W.Q_E)
    assert 0.8e-4 < c4.charge_pos.std() < 1.2e-4


def test_bench_reads_its_roofline_constants_from_the_committed_tables():
    """bench.py takes flop per pair and DRAM bytes per launch from profiles/*.md (ncu tables): every case it looks up must
    be there and sane, or the driver's bench run would die on the GPU box."""
    import importlib.util
    import os
    root = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
    spec = importlib.util.spec_from_file_location("bench_module", os.path.join(root, "bench.py"))
    bench = importlib.util.module_from_spec(spec)
    spec.loader.exec_module(bench)
    ops = bench.load_opcounts()
    need = ["eval_rect_uniform", "eval_rect_single", "eval_images", "eval_images_single", "eval_tri_uniform", "eval_wire",
            "assemble_c2", "assemble_images", "charges"]
    for case in need:
        assert case in ops, case
        o = ops[case]
        assert 10.0 < o["flop"] < 400.0 and 5.0 < o["fp64_instr"] < 250.0
        assert abs(o["flop"] - (2 * o["dfma"] + o["dmul"] + o["dadd"])) < 1e-9
    for pair, single in bench.ELEMENTWISE_CASE.items():
        assert ops[single]["flop"] > ops[pair]["flop"]                 # sharing an edge saves work, never adds
    traffic = bench.load_bench_traffic()
    for kern in ("eval_kernel", "assemble_kernel", "gemm_kernel"):
        assert traffic[("C2", kern)] > 1e6
    from workloads import configs as W
    fl, inst = bench.flop_per_pair(W.thgem(d=10, n_plane=6, n_grid=2), ops)
    assert ops["eval_tri_uniform"]["flop"] <= fl <= ops["eval_rect_uniform"]["flop"] and inst < fl


def test_no_alloc_test_file_is_collected_last():
    """tests/test_zz_no_alloc.py must stay the last file pytest collects (alphabetical order): the suite runs with
    `pytest -x`, and a failure in that file must not hide any other test."""
    import glob
    import os
    here = os.path.dirname(os.path.abspath(__file__))
    files = sorted(os.path.basename(p) for p in glob.glob(os.path.join(here, "test_*.py")))
    assert files[-1] == "test_zz_no_alloc.py", files
