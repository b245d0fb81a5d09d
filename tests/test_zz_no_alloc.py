"""bs_vdot_noalloc (include/bs.h): the variant of bs_vdot whose scratch is a static __device__ array, for callers that
cannot call cudaMalloc.  Collected LAST (file name) so that a failure here hides no other test under `pytest -x`.

Checked against the existing path (bs_vdot, malloc'ed scratch) on two calls in a row with different inputs -- the second
call finds the first call's partials in the shared array -- at a size that spans several tiles and a ragged tail, then at
a size of one partial tile, zero length, and beyond the stated maximum (must be refused, not truncated).
Tolerance: the energies' bar of the other tests (1e-10 absolute) tightened to 1e-12, the two paths differ only in the
order of a 1e6-term sum of O(1e-6) products.
"""
import numpy as np
import pytest

import synth_inputs as si

pytestmark = pytest.mark.gpu


def test_vdot_noalloc_matches_bs_vdot_twice_in_a_row():
    import torch
    from paper_2606_28952_b200 import bs
    sec = bs.bs_sector_build(12, 6, 5)                     # dim 731,808 = 11 tiles of 65,536 + a tail of 10,912
    assert sec.dim == 924 * 792 and sec.dim % 65536 != 0
    bs.bs_noalloc_setup()
    assert bs.bs_noalloc_max_dim() == 8192 * 65536
    res = torch.zeros(1, dtype=torch.complex128, device="cuda")
    # call 1: long vectors (fills 12 partials); call 2: other data; both against the existing path
    pairs = [(si.random_state(sec.dim, 5), si.random_state(sec.dim, 6)),
             (si.random_state(sec.dim, 7), si.random_state(sec.dim, 8))]
    for a_np, b_np in pairs:
        a, b = torch.from_numpy(a_np).cuda(), torch.from_numpy(b_np).cuda()
        want = bs.bs_vdot(sec, a, b)
        bs.bs_vdot_noalloc(a, b, res)
        got = complex(res.cpu()[0])
        assert abs(got - want) <= 1e-12, (got, want)
        assert abs(got - np.vdot(a_np, b_np)) <= 1e-12
        bs.bs_vdot_noalloc(a, b, res)                      # same inputs again: deterministic, bit for bit
        assert complex(res.cpu()[0]) == got
    # a SHORT vector right after a long one: the stale partials of the long call must not leak in
    small = bs.bs_sector_build(6, 3, 3)                    # 400 amplitudes: one partial tile
    a_np, b_np = si.random_state(400, 1), si.random_state(400, 2)
    a, b = torch.from_numpy(a_np).cuda(), torch.from_numpy(b_np).cuda()
    bs.bs_vdot_noalloc(a, b, res)
    assert abs(complex(res.cpu()[0]) - bs.bs_vdot(small, a, b)) <= 1e-12
    # zero length: (0, 0), whatever the array holds
    empty = torch.zeros(0, dtype=torch.complex128, device="cuda")
    res.fill_(7.0)
    rc = bs._lib.bs_vdot_noalloc(a.data_ptr(), b.data_ptr(), 0, res.data_ptr(), None)
    torch.cuda.synchronize()
    assert rc == 0 and complex(res.cpu()[0]) == 0
    del empty
    # beyond the static scratch: refused with a clear error, result untouched
    res.fill_(3.0)
    rc = bs._lib.bs_vdot_noalloc(a.data_ptr(), b.data_ptr(), bs.bs_noalloc_max_dim() + 1, res.data_ptr(), None)
    assert rc == bs.BS_ERR_ARG and "exceed the static scratch" in bs.bs_last_error()
    torch.cuda.synchronize()
    assert complex(res.cpu()[0]) == 3.0


def test_vdot_noalloc_allocates_nothing():
    """Device memory in use does not change across calls (the first call above or here did the one-off set-up)."""
    import torch
    from paper_2606_28952_b200 import bs
    bs.bs_noalloc_setup()
    n = 1 << 20
    a = torch.from_numpy(si.random_state(n, 3)).cuda()
    b = torch.from_numpy(si.random_state(n, 4)).cuda()
    res = torch.zeros(1, dtype=torch.complex128, device="cuda")
    bs.bs_vdot_noalloc(a, b, res)
    torch.cuda.synchronize()
    free0, _ = torch.cuda.mem_get_info()
    for _ in range(5):
        bs.bs_vdot_noalloc(a, b, res)
    torch.cuda.synchronize()
    free1, _ = torch.cuda.mem_get_info()
    assert free1 == free0
    assert abs(complex(res.cpu()[0]) - np.vdot(a.cpu().numpy(), b.cpu().numpy())) <= 1e-12
