"""CPU-side checks of the C-ABI library: it loads, exports every symbol include/heget.h declares, validates its
arguments and reports errors through status codes -- no compute call is made (there is no GPU here).

Also the host logic that needs no device: the process generator's counts (Table 1), the colour matrix
the plug-in carries against the oracle's brute-force matrix (eq. 9; Table 4), and the
event sharding of SURVEY.md 8(e).
"""
import ctypes as C
import os
import re

import numpy as np
import pytest

import paper_0909_5257_b200 as hg
from paper_0909_5257_b200 import build as hbuild

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
    assert lib.heget_process_create(b"g g > g g g g g g g", 500.0, 0.118, None, 0, C.byref(h)) == hg.EUNSUPPORTED
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


def test_shard_range_partitions_events():
    for n, world in [(2 ** 20, 8), (1000, 3), (5, 8), (0, 2)]:
        parts = [hg.shard_range(n, r, world) for r in range(world)]
        assert parts[0][0] == 0 and sum(c for _, c in parts) == n
        for (lo, c), (lo2, _) in zip(parts, parts[1:]):
            assert lo + c == lo2
