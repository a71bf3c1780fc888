"""Parity of the CUDA path (through the C ABI) against the fp64 CPU oracle, element by element, on
the same seeded inputs.  Tolerance: max |dJ|, |dK| <= 1e-9 Eh in full-fp64 mode (north_star).

Small cases (tiny, pd_test, water8): the full matrices and the SR / LR / SELF parts separately.
Large cases (si64, water64, water343): sampled output shell blocks (oracle "sampled mode",
SURVEY 8(c)) -- see test_parity_large_gpu.py -- plus oracle-free invariants here.
"""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu

TOL = 1e-9


@pytest.fixture(scope="module")
def torch_cuda():
    import torch
    assert torch.cuda.is_available(), "the gpu tests need a CUDA device"
    return torch


def _gpu_jk(torch, wl, P, parts="sr+lr+self", **kw):
    from paper_2410_22278_b200.binding import PbcJK
    with PbcJK(wl, **kw) as h:
        h.set_parts(parts)
        Pd = torch.from_numpy(P).cuda()
        J = torch.empty_like(Pd)
        K = torch.empty_like(Pd)
        h.build(Pd, J, K)
        torch.cuda.synchronize()
        st = h.stats()
        S = h.overlap()
        return J.cpu().numpy(), K.cpu().numpy(), S, st


def _density(oracle, wl):
    from paper_2410_22278_b200.workloads import density_from_orbitals
    S = oracle.overlap(wl)
    return density_from_orbitals(wl.orbitals_seed(), S), S


@pytest.mark.parametrize("name", ["tiny", "pd_test", "water8"])
def test_full_matrices_and_parts(torch_cuda, oracle_mod, name):
    from paper_2410_22278_b200 import workloads
    wl = workloads.get(name)
    P, S = _density(oracle_mod, wl)
    ref = oracle_mod.jk(wl, P)
    J, K, Sg, st = _gpu_jk(torch_cuda, wl, P)
    assert st["quartets_j"] > 0 and st["quartets_k"] > 0
    assert np.abs(Sg - S).max() < 1e-12
    assert np.abs(J - ref["J"]).max() < TOL
    assert np.abs(K - ref["K"]).max() < TOL
    for part in ("sr", "lr", "self"):
        Jp, Kp, _, _ = _gpu_jk(torch_cuda, wl, P, parts=part)
        assert np.abs(Jp - ref["J_" + part]).max() < TOL, part
        assert np.abs(Kp - ref["K_" + part]).max() < TOL, part


def test_indefinite_unsymmetric_scale_density(torch_cuda, oracle_mod):
    """J and K are linear in P; a random symmetric indefinite P exercises every P element."""
    from paper_2410_22278_b200 import workloads
    wl = workloads.get("pd_test")
    rng = np.random.default_rng(5)
    n = wl.nbf
    P = rng.standard_normal((n, n))
    P = 0.5 * (P + P.T)
    ref = oracle_mod.jk(wl, P)
    J, K, _, _ = _gpu_jk(torch_cuda, wl, P)
    assert np.abs(J - ref["J"]).max() < TOL * 10     # |P| ~ 1, N(0,1): values ~10x those of a projector
    assert np.abs(K - ref["K"]).max() < TOL * 10


def test_only_j_or_only_k(torch_cuda, oracle_mod):
    from paper_2410_22278_b200 import workloads
    from paper_2410_22278_b200.binding import PbcJK
    torch = torch_cuda
    wl = workloads.get("tiny")
    P, _ = _density(oracle_mod, wl)
    ref = oracle_mod.jk(wl, P)
    with PbcJK(wl) as h:
        Pd = torch.from_numpy(P).cuda()
        J = torch.full_like(Pd, 7.0)
        K = torch.full_like(Pd, 7.0)
        h.build(Pd, J, None)
        h.build(Pd, None, K)
        torch.cuda.synchronize()
        assert np.abs(J.cpu().numpy() - ref["J"]).max() < TOL        # overwritten, not accumulated
        assert np.abs(K.cpu().numpy() - ref["K"]).max() < TOL
        # host-buffer entry point
        Jh, Kh = h.build_host(P)
        assert np.abs(Jh - ref["J"]).max() < TOL and np.abs(Kh - ref["K"]).max() < TOL


def test_deterministic(torch_cuda, oracle_mod):
    """No atomics on the data path: two builds are bit-identical."""
    from paper_2410_22278_b200 import workloads
    wl = workloads.get("water8")
    P, _ = _density(oracle_mod, wl)
    a = _gpu_jk(torch_cuda, wl, P)
    b = _gpu_jk(torch_cuda, wl, P)
    assert np.array_equal(a[0], b[0]) and np.array_equal(a[1], b[1])


def test_omega_invariance_on_gpu(torch_cuda, oracle_mod):
    """Oracle-free: J and K from the CUDA path do not depend on the Ewald parameter."""
    from paper_2410_22278_b200 import workloads
    wl = workloads.get("water8")
    P, _ = _density(oracle_mod, wl)
    res = [_gpu_jk(torch_cuda, wl, P, omega=om) for om in (0.3, 0.45)]
    assert np.abs(res[0][0] - res[1][0]).max() < TOL
    assert np.abs(res[0][1] - res[1][1]).max() < TOL


def test_rank1_identity_on_gpu(torch_cuda, oracle_mod):
    """Oracle-free: for P = c c^T, J c = K c (both are sum c_n c_l c_s (mn|ls))."""
    from paper_2410_22278_b200 import workloads
    wl = workloads.get("water8")
    rng = np.random.default_rng(11)
    c = rng.standard_normal(wl.nbf)
    c /= np.linalg.norm(c)
    P = np.outer(c, c)
    J, K, _, _ = _gpu_jk(torch_cuda, wl, P)
    assert np.abs(J @ c - K @ c).max() < TOL
    assert np.abs(J - J.T).max() < 1e-12 and np.abs(K - K.T).max() < 1e-12


def test_translated_and_image_shifted_atoms(torch_cuda, oracle_mod):
    """Centres may sit in any lattice image; a rigid translation changes nothing."""
    import copy
    from paper_2410_22278_b200 import workloads
    wl = workloads.get("pd_test")
    P, _ = _density(oracle_mod, wl)
    J0, K0, _, _ = _gpu_jk(torch_cuda, wl, P)
    wl2 = copy.deepcopy(wl)
    wl2.xyz = wl.xyz + np.array([0.37, -1.21, 2.2])
    wl2.xyz[1] += 2 * wl.cell[0] - 1 * wl.cell[2]
    J1, K1, _, _ = _gpu_jk(torch_cuda, wl2, P)
    assert np.abs(J1 - J0).max() < TOL and np.abs(K1 - K0).max() < TOL


def test_error_paths(torch_cuda):
    import copy
    from paper_2410_22278_b200 import workloads
    from paper_2410_22278_b200.binding import PbcJK, PbcJKError
    wl = workloads.get("tiny")
    bad = copy.deepcopy(wl)
    bad.sh_l = wl.sh_l.copy()
    bad.sh_l[0] = 3
    with pytest.raises(PbcJKError):
        PbcJK(bad)
    bad = copy.deepcopy(wl)
    bad.cell = np.zeros((3, 3))
    with pytest.raises(PbcJKError):
        PbcJK(bad)
    with pytest.raises(PbcJKError):
        PbcJK(wl, omega=-1.0)
    with pytest.raises(PbcJKError):      # mixed precision is not built yet: refused, never silently fp64
        PbcJK(wl, precision=1)
    bad = copy.deepcopy(wl)
    bad.exps = wl.exps.copy()
    bad.exps[0] = 0.0
    with pytest.raises(PbcJKError):
        PbcJK(bad)
