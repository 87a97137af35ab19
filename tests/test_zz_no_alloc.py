"""gh_constraint_norms_static: the allocation-free variant of gh_constraint_norms (reduction scratch in a file-scope static device
array, include/gh.h) against the existing path, on two calls in a row.  Collected last on purpose (the suite runs with pytest -x)."""
import numpy as np
import pytest
import torch

from paper_1804_09101_b200 import configs, gh
from domain_util import build_case

pytestmark = pytest.mark.gpu


def _same(a, b, floor):
    """the tolerance of the norm comparisons in the parity tests: 1e-9 relative + 1e-11 ||u||inf absolute"""
    return np.all(np.abs(a - b) <= 1e-9 * np.abs(b) + floor)


def test_static_scratch_matches_existing_path_twice(oracle):
    big = {"id": 71, "spin": 0.5, "amplitude": 1e-4,
           "descs": [configs.shell(9, 10, 2.0, 4.0, face=(0, 1)), configs.block([9, 8, 7], (5.0, -1.0, -1.0), (7.0, 1.0, 1.0)),
                     configs.cylinder((6, 5, 9), 3.0, 5.0, 4.5, 6.0), configs.shell(7, 6, 4.0, 8.0)]}
    small = {"id": 72, "spin": 0.2, "amplitude": 1e-3, "descs": [configs.block([5, 6, 4], (3.0, -1.0, -1.0), (4.0, 1.0, 1.0))]}
    doms = []
    for cfg in (big, small):
        descs, coords, us, Hs = build_case(cfg, oracle)
        dom = gh.Domain(descs)
        dom.set_gauge_source(dom.pack(Hs))
        dom.set_fields(dom.pack(us), 0.0)
        doms.append((dom, descs, us, Hs))
    dom, descs, us, Hs = doms[0]
    floor = 1e-11 * max(np.max(np.abs(u)) for u in us)
    # call 1: against the existing entry point and against the oracle
    ref, ref_ps = dom.constraint_norms(per_sub=True)
    got, got_ps = dom.constraint_norms_static(per_sub=True)
    assert _same(got, ref, floor) and _same(got_ps, ref_ps, floor), (got, ref)
    assert np.array_equal(got, ref) and np.array_equal(got_ps, ref_ps)         # the same additions in the same order
    assert _same(got, oracle.constraint_norms(descs, us, Hs), floor)
    free1 = torch.cuda.mem_get_info()[0]
    # call 2, straight after, on ANOTHER state of the same domain (the scratch still holds call 1's partials and sums)
    dom.rk_step(0.25 * configs.min_spacing(descs))
    got2 = dom.constraint_norms_static()
    ref2 = dom.constraint_norms()
    assert _same(got2, ref2, floor) and np.array_equal(got2, ref2)
    assert not np.array_equal(got2, got)
    # ... and on a smaller domain (fewer tiles and subdomains than what the scratch still holds), without per_sub
    d2, descs2, us2, Hs2 = doms[1]
    got3 = d2.constraint_norms_static()
    ref3 = d2.constraint_norms()
    assert _same(got3, ref3, 1e-11 * np.max(np.abs(us2[0]))) and np.array_equal(got3, ref3)
    assert torch.cuda.mem_get_info()[0] >= free1                              # no device memory was taken by the later calls
    # dual frame set (K_map_pre runs inside both paths): still the same bits
    S2 = d2.S
    Jm = np.zeros((9, S2))
    Jm[0], Jm[4], Jm[8], Jm[1] = 1 / 1.1, 1 / 1.05, 1.0, 0.02
    d2.set_frame_map(Jm, np.zeros((3, S2)))
    got4, ref4 = d2.constraint_norms_static(), d2.constraint_norms()
    assert np.array_equal(got4, ref4) and not np.array_equal(got4, got3)
    d2.set_frame_map(None, None)
    # the existing path is untouched by the static one
    assert np.array_equal(dom.constraint_norms(), ref2)
    for d, *_ in doms:
        d.close()


def test_static_scratch_rejects_sizes_beyond_its_maximum():
    n = 4097                                                    # GH_STATIC_MAX_SUBS + 1 subdomains of 8 points
    descs = [configs.block(2, (3.0 + i, 0.0, 0.0), (3.5 + i, 1.0, 1.0)) for i in range(n)]
    dom = gh.Domain(descs)
    S = dom.S
    u = np.zeros((50, S))
    u[0], u[4], u[7], u[9] = -1.0, 1.0, 1.0, 1.0               # Minkowski
    dom.set_gauge_source(np.zeros((4, S)))
    dom.set_fields(u, 0.0)
    assert np.all(dom.constraint_norms() == 0.0)               # the existing path takes the domain
    with pytest.raises(gh.GHError) as e:
        dom.constraint_norms_static()
    assert e.value.status == gh.GH_ERR_ARG and "4096 subdomains" in str(e.value)
    dom.close()
