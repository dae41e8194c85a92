"""CPU-side checks of the C-ABI library: it loads, exports every symbol include/heget.h declares, validates its
arguments and reports errors through status codes -- no compute call is made (there is no GPU here).

Also the host logic that needs no device: the process generator's counts (Table 1), the colour matrix
the plug-in carries against the oracle's brute-force matrix (eq. 9; Table 4), and the
event sharding of SURVEY.md 8(e).
"""
import ctypes as C
import math
import os
import re

import numpy as np
import pytest

import paper_0909_5257_b200 as hg
from paper_0909_5257_b200 import build as hbuild
from golden_io import rows

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def lib():
    hbuild.build_library()
    hbuild.build_kernels(["u u~ > g g", "g g > g g", "u u > u u", "g g > g g g", "u u > u u g g"], verbose=False)
    return hg.lib()


def test_exports_every_declared_symbol(lib):
    text = open(os.path.join(ROOT, "include", "heget.h")).read()
    text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)
    declared = set(re.findall(r"\b(heget_[a-z0-9_]+)\s*\(", text))
    assert declared == set(hg.EXPORTS)
    for name in declared:
        assert getattr(lib, name) is not None


def test_argument_validation(lib):
    h = C.c_void_p()
    assert lib.heget_process_create(None, 500.0, 0.118, None, 0, C.byref(h)) == hg.EINVAL
    assert b"NULL" in lib.heget_last_error()
    assert lib.heget_process_create(b"u u~ > g g", -1.0, 0.118, None, 0, C.byref(h)) == hg.EINVAL
    assert lib.heget_process_create(b"u u~ > g g", 500.0, 0.0, None, 0, C.byref(h)) == hg.EINVAL
    assert lib.heget_process_create(b"u u~ > g g", 500.0, 0.118, None, 7, C.byref(h)) == hg.EINVAL
    assert lib.heget_process_create(b"u u~ > g g", 500.0, 0.118, None, 0, None) == hg.EINVAL
    assert lib.heget_process_create(b"U U~ > G G", 500.0, 0.118, None, 0, C.byref(h)) == hg.EINVAL
    assert lib.heget_process_info(None, None) == hg.EINVAL
    assert lib.heget_sample_momenta(None, 0, 0, 16, None, None, None, None) == hg.EINVAL
    assert lib.heget_eval_me2(None, None, 16, 0, None, 0, 0, None, None) == hg.EINVAL
    assert lib.heget_run_host(None, 0, 0, 16, None, None, None, 0, None, None, None) == hg.EINVAL
    lib.heget_destroy(None)      # allowed


def test_unsupported_process(lib, tmp_path, monkeypatch):
    monkeypatch.setenv("HEGET_CACHE_DIR", str(tmp_path))
    h = C.c_void_p()
    # syntactically fine, but not massless QCD
    assert lib.heget_process_create(b"e+ e- > u u~", 500.0, 0.118, None, 0, C.byref(h)) == hg.EINVAL   # '+' is not a tag character
    assert lib.heget_process_create(b"z g > g g", 500.0, 0.118, None, 0, C.byref(h)) == hg.EUNSUPPORTED
    assert b"unsupported particle" in lib.heget_last_error()
    # QCD, but no tree diagram conserves flavour
    assert lib.heget_process_create(b"u u > g g", 500.0, 0.118, None, 0, C.byref(h)) == hg.EUNSUPPORTED
    assert lib.heget_process_create(b"g g > g g g g g g", 500.0, 0.118, None, 0, C.byref(h)) == hg.EUNSUPPORTED      # 8 legs
    with pytest.raises(hg.HegetError) as ei:
        hg.Process("u > g g", 500.0)
    assert ei.value.status in (hg.EINVAL, hg.EUNSUPPORTED)


def test_handle_calls_without_device(lib):
    P = hg.Process("u u~ > g g", 500.0)
    i = P.info
    assert (i.n_ext, i.n_hel, i.n_hel_eval, i.n_diagrams, i.n_color) == (4, 16, 8, 3, 2)
    assert i.avg_spin == 0.25 and i.avg_color == 1.0 / 9.0 and i.sym_factor == 0.5
    assert i.flops_per_event > 0
    # zero events is a no-op that needs neither pointers nor a device
    assert lib.heget_sample_momenta(P._h, 0, 0, 0, None, None, None, None) == hg.OK
    assert lib.heget_eval_me2(P._h, None, 0, 0, None, 0, 0, None, None) == hg.OK
    assert lib.heget_run_host(P._h, 0, 0, 0, None, None, None, 0, None, None, None) == hg.OK
    # required pointers
    assert lib.heget_sample_momenta(P._h, 0, 0, 8, None, None, None, None) == hg.EINVAL
    assert lib.heget_eval_me2(P._h, None, 8, 0, None, 0, 0, None, None) == hg.EINVAL
    assert lib.heget_eval_me2(P._h, None, 8, 9, None, 0, 0, None, None) == hg.EINVAL
    assert lib.heget_eval_me2(P._h, None, 8, hg.HEL_FIXED, None, 0, 0, None, None) == hg.EINVAL
    assert lib.heget_set_lanes(P._h, 3) == hg.EINVAL
    assert P.info.lanes_wide == 8            # 8 non-vanishing helicity configurations
    assert lib.heget_set_lanes(P._h, 8) == hg.OK and lib.heget_set_lanes(P._h, 1) == hg.OK and lib.heget_set_lanes(P._h, 0) == hg.OK
    P.close()
    P.close()


TABLE1 = {   # (diagrams, colour bases): Table 1, PAPER.md:39-47 (conventions A11, A12 of DESIGN.md)
    "u u~ > g g": (3, 2), "g g > g g": (6, 6), "u u > u u": (2, 2),
    "g g > g g g": (45, 24), "u u > u u g g": (76, 40),
}


@pytest.mark.parametrize("name", sorted(TABLE1))
def test_generator_counts_and_colour_matrix(lib, oracle_process, name):
    P = hg.Process(name, 1000.0)
    assert (P.info.n_diagrams, P.info.n_color) == TABLE1[name]
    Cg = P.color_matrix(0).numpy()
    Co = oracle_process(name).colour_matrix()
    assert Cg.shape == Co.shape
    assert np.allclose(Cg, Cg.T, atol=0)
    # the two bases may be enumerated in different orders: compare what is unique -- the spectrum and the multiset of entries
    assert np.allclose(np.sort(np.linalg.eigvalsh(Cg)), np.sort(np.linalg.eigvalsh(Co)), atol=1e-10)
    assert np.allclose(np.sort(Cg.ravel()), np.sort(Co.ravel()), atol=1e-12)
    # the reduced matrix the kernel contracts is a congruence of C: it has the same rank as C restricted to what the diagrams span
    Cr = P.color_matrix(1).numpy()
    assert Cr.shape[0] == P.info.n_color_reduced <= P.info.n_color_eval
    assert np.allclose(Cr, Cr.T, atol=1e-12)
    assert np.linalg.eigvalsh(Cr).min() > -1e-10


# ---- the table back end (no compiler, no device needed to build and inspect a process) ---------------------------------------

@pytest.mark.parametrize("row", rows("table1_counts.txt"), ids=lambda r: r[0])
def test_table_generator_reproduces_table1_and_table4(lib, row):
    """The generator's table program against the paper's own numbers (Tables 1 and 4) for all twelve
    processes -- including g g -> 5g and u u -> u u g g g, which the paper could not run or only barely ran.
    The merged currents and centroid closings of the table back end must still count every Feynman diagram exactly once."""
    name, n_diag, n_col = row[0], int(row[1]), int(row[2])
    distinct = {r[0]: int(r[1]) for r in rows("table4_distinct.txt")}[name]
    P = hg.Process(name, 1000.0, kernel="table")
    i = P.info
    assert i.kernel == hg.KERNEL_TABLE
    assert (i.n_diagrams, i.n_color) == (n_diag, n_col)
    Cp = P.color_matrix(0).numpy()
    assert Cp.shape == (n_col, n_col) and np.array_equal(Cp, Cp.T)
    vals = np.unique(np.round(Cp[np.abs(Cp) > 1e-12], 9))
    assert len(vals) == distinct
    # the accumulated basis spans what the diagrams span: its matrix is a congruence of C, and its dimension is (n-2)! for
    # pure gluons (the f-basis); its rank cannot exceed the colour rank
    Ca = P.color_matrix(2).numpy()
    assert Ca.shape[0] == i.n_color_accum <= i.n_color_reduced <= i.n_color_eval <= i.n_color
    assert np.allclose(Ca, Ca.T, atol=1e-12) and np.linalg.eigvalsh(Ca).min() > -1e-9       # positive semi-definite (u u -> u u g g g: 48 elements, rank 46)
    assert np.linalg.matrix_rank(Ca, tol=1e-9) <= i.color_rank <= i.n_color
    if "u" not in name:
        assert i.n_color_accum == math.factorial(i.n_ext - 2)
        # the trace bases of 4, 5, 6 gluons are independent; with 7 gluons the 720 single traces are no longer
        # independent for N = 3 (the generator finds rank 656)
        assert i.color_rank == n_col or i.n_ext == 7
    P.close()


def test_colour_rank_matches_survey_a13(lib):
    """the paper's over-complete two-quark-line bases have rank 2 / 4 / 12 / 46 of 2 / 8 / 40 / 240."""
    for name, rank in [("u u > u u", 2), ("u u > u u g", 4), ("u u > u u g g", 12), ("u u > u u g g g", 46), ("u u~ > g g g", 6)]:
        P = hg.Process(name, 1000.0, kernel="table")
        assert P.info.color_rank == rank
        assert np.linalg.matrix_rank(P.color_matrix(0).numpy(), tol=1e-9) == rank
        P.close()


def test_table_and_straight_back_ends_describe_the_same_process(lib):
    for name in ["u u~ > g g", "g g > g g g", "u u > u u g g"]:
        A = hg.Process(name, 1000.0, kernel="straight"); B = hg.Process(name, 1000.0, kernel="table")
        a, b = A.info, B.info
        assert (a.kernel, b.kernel) == (hg.KERNEL_STRAIGHT, hg.KERNEL_TABLE)
        for f in ("n_ext", "n_hel", "n_hel_eval", "n_diagrams", "n_topologies", "n_color", "n_color_eval", "n_color_reduced", "avg_spin", "avg_color", "sym_factor"):
            assert getattr(a, f) == getattr(b, f), f
        assert np.array_equal(A.color_matrix(0).numpy(), B.color_matrix(0).numpy())
        assert b.flops_per_event < a.flops_per_event      # helicity recycling + merged currents: fewer flops for the same sum
        # switching a handle back and forth keeps it usable
        A.set_kernel("table"); assert A.info.kernel == hg.KERNEL_TABLE
        A.set_kernel("auto"); assert A.info.kernel == hg.KERNEL_STRAIGHT
        A.close(); B.close()
    P = hg.Process("g g > g g g g", 1500.0)
    assert P.info.kernel == hg.KERNEL_TABLE and P.info.lanes == 32       # AUTO: the big processes take the table back end
    assert lib.heget_set_lanes(P._h, 1) == hg.EINVAL and lib.heget_set_lanes(P._h, 0) == hg.OK
    assert lib.heget_set_kernel(P._h, 7) == hg.EINVAL and lib.heget_set_kernel(None, 0) == hg.EINVAL
    P.close()


def test_shard_range_partitions_events():
    for n, world in [(2 ** 20, 8), (1000, 3), (5, 8), (0, 2)]:
        parts = [hg.shard_range(n, r, world) for r in range(world)]
        assert parts[0][0] == 0 and sum(c for _, c in parts) == n
        for (lo, c), (lo2, _) in zip(parts, parts[1:]):
            assert lo + c == lo2
