"""The allocation-free entry point `pbc_jk_overlap_noalloc` (include/pbc_jk.h): the overlap S (eq 21)
recomputed into a caller's device buffer with the scratch stack in a file-scope device array of the library.

Checked against the existing path (`pbc_jk_overlap`, the S formed at create in cudaMalloc'ed workspaces), within the
tolerance of the parity tests, on two calls in a row -- the second call finds the first call's contents in the shared
scratch -- and after a call on ANOTHER handle has left a different system's values there.  Collected last on purpose
(the suite runs with `pytest -x`).  Passes alone in a fresh process and after the other tests: it uses nothing but
its own handles."""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu

TOL = 1e-9        # the fp64 tolerance of tests/test_parity_gpu.py; the two paths run the same kernels: observed 0.0


def _handle(name):
    from paper_2410_22278_b200 import workloads
    from paper_2410_22278_b200.binding import PbcJK
    wl = workloads.get(name)
    return wl, PbcJK(wl)


def _call(h, torch, fill):
    S = torch.full((h.nbf, h.nbf), fill, dtype=torch.float64, device="cuda")
    h.overlap_noalloc(S)
    torch.cuda.synchronize()
    return S.cpu().numpy()


def test_overlap_noalloc_matches_existing_path_twice():
    import torch
    wl, h = _handle("water8")                     # N = 200: s, p and d shells, padded to 256 inside
    S_ref = h.overlap()
    assert np.isfinite(S_ref).all() and abs(np.diag(S_ref) - 1.0).max() < 0.5
    S1 = _call(h, torch, float("nan"))
    S2 = _call(h, torch, 7.0)
    assert np.isfinite(S1).all() and np.isfinite(S2).all()
    assert abs(S1 - S_ref).max() <= TOL
    assert abs(S2 - S_ref).max() <= TOL
    assert np.array_equal(S1, S2)                 # the shared scratch is cleared per call: no carry-over


def test_overlap_noalloc_other_handle_in_between():
    """The array is shared by every handle: a smaller system's call in between must not leak into the next one."""
    import torch
    wl_a, ha = _handle("water8")
    wl_b, hb = _handle("pd_test")                 # N = 14, another cell: leaves its values at the front of the scratch
    Sa_ref, Sb_ref = ha.overlap(), hb.overlap()
    Sa1 = _call(ha, torch, float("nan"))
    Sb = _call(hb, torch, float("nan"))
    Sa2 = _call(ha, torch, float("nan"))
    assert abs(Sb - Sb_ref).max() <= TOL
    assert abs(Sa1 - Sa_ref).max() <= TOL and abs(Sa2 - Sa_ref).max() <= TOL
    assert np.array_equal(Sa1, Sa2)


def test_overlap_noalloc_allocates_nothing_and_rejects_large():
    import torch
    from paper_2410_22278_b200.binding import PbcJKError
    wl, h = _handle("water8")
    S = torch.empty((h.nbf, h.nbf), dtype=torch.float64, device="cuda")
    h.overlap_noalloc(S)                          # warm: module and kernels loaded
    torch.cuda.synchronize()
    free0, _ = torch.cuda.mem_get_info()
    for _ in range(3):
        h.overlap_noalloc(S)
    torch.cuda.synchronize()
    free1, _ = torch.cuda.mem_get_info()
    assert free1 == free0                         # driver-level free memory unchanged: nothing was allocated
    # beyond the static scratch (N padded to 64 > 512): refused with a clear text, output untouched
    wl_big, hb = _handle("si64")                  # N = 960
    Sb = torch.full((hb.nbf, hb.nbf), 3.0, dtype=torch.float64, device="cuda")
    with pytest.raises(PbcJKError) as ei:
        hb.overlap_noalloc(Sb)
    assert "static scratch" in str(ei.value) and "512" in str(ei.value)
    torch.cuda.synchronize()
    assert float(Sb.min()) == 3.0 and float(Sb.max()) == 3.0
