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
    # an atom given thousands of cells away (far outside the packed image range if it were not folded back)
    wl3 = copy.deepcopy(wl)
    wl3.xyz[0] += 3000 * wl.cell[1] - 2500 * wl.cell[0]
    J2, K2, _, _ = _gpu_jk(torch_cuda, wl3, P)
    assert np.abs(J2 - J0).max() < TOL and np.abs(K2 - K0).max() < TOL


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
    with pytest.raises(PbcJKError):      # 0 = fp64, 1 = mixed; anything else is refused
        PbcJK(wl, precision=2)
    # a cell far too small for the exponents: the lattice indices of the real-space sums would leave the packed
    # 10-bit range -> PBC_JK_ERR_UNSUPPORTED at create, never a silent wrap-around
    bad = copy.deepcopy(wl)
    bad.cell = wl.cell * 0.004
    bad.xyz = wl.xyz * 0.004
    bad.r_cut = 0.0
    with pytest.raises(PbcJKError) as ei:
        PbcJK(bad)
    assert ei.value.code == -4
    bad = copy.deepcopy(wl)
    bad.sh_off = wl.sh_off.copy()
    bad.sh_off[0] = -1
    with pytest.raises(PbcJKError):
        PbcJK(bad)
    bad = copy.deepcopy(wl)
    bad.exps = wl.exps.copy()
    bad.exps[0] = 0.0
    with pytest.raises(PbcJKError):
        PbcJK(bad)


def test_odd_g_batch(torch_cuda, oracle_mod):
    """The reciprocal-space batch size is a free parameter: an odd, small value (ragged last batch, slot padding)
    gives the same LR part as the default and as the oracle."""
    from paper_2410_22278_b200 import workloads
    wl = workloads.get("water8")
    P, _ = _density(oracle_mod, wl)
    ref = oracle_mod.jk(wl, P, parts="lr+self")
    J0, K0, _, _ = _gpu_jk(torch_cuda, wl, P, parts="lr+self")
    for nb in (7, 33):
        J, K, _, _ = _gpu_jk(torch_cuda, wl, P, parts="lr+self", lr_g_batch=nb)
        assert np.abs(J - ref["J"]).max() < TOL and np.abs(K - ref["K"]).max() < TOL, nb
        assert np.abs(J - J0).max() < 1e-11 and np.abs(K - K0).max() < 1e-11, nb


def test_profile_mode_is_bit_identical(torch_cuda, oracle_mod):
    """Serial class launches (profile mode) and the forked internal streams accumulate every output block in the same
    order: same bits."""
    from paper_2410_22278_b200 import workloads
    from paper_2410_22278_b200.binding import PbcJK
    torch = torch_cuda
    wl = workloads.get("water8")
    P, _ = _density(oracle_mod, wl)
    with PbcJK(wl) as h:
        Pd = torch.from_numpy(P).cuda()
        J0, K0, J1, K1 = (torch.empty_like(Pd) for _ in range(4))
        h.build(Pd, J0, K0)
        h.set_profile(True)
        h.build(Pd, J1, K1)
        torch.cuda.synchronize()
        cs = h.class_stats()
        assert len(cs) > 10 and all(c["ms"] > 0 for c in cs)
        assert torch.equal(J0, J1) and torch.equal(K0, K1)
        h.set_profile(False)
        h.build(Pd, J1, K1)
        torch.cuda.synchronize()
        assert all(c["ms"] == 0 for c in h.class_stats())      # no stale event reads after a non-profiled build
        st = h.stats()
        assert st["ms_sr_k"] > 0 and st["ms_sr_j"] > 0


def test_shards_sum_to_full_build(torch_cuda, oracle_mod):
    """pbc_jk_set_shard(r, n): the n partial J and K (real-space blocks / bras and G batches dealt round-robin, SELF on
    rank 0) add up to the full matrices -- what the one all-reduce of the multi-GPU build sums."""
    from paper_2410_22278_b200 import workloads
    from paper_2410_22278_b200.binding import PbcJK
    torch = torch_cuda
    wl = workloads.get("water8")
    P, _ = _density(oracle_mod, wl)
    ref = oracle_mod.jk(wl, P)
    Pd = torch.from_numpy(P).cuda()
    n = 3
    Js, Ks = torch.zeros_like(Pd), torch.zeros_like(Pd)
    quart = 0
    for r in range(n):
        with PbcJK(wl, lr_g_batch=16) as h:
            h.set_shard(r, n)
            J, K = torch.empty_like(Pd), torch.empty_like(Pd)
            h.build(Pd, J, K)
            torch.cuda.synchronize()
            quart += h.stats()["quartets_k"]
            Js += J
            Ks += K
    with PbcJK(wl, lr_g_batch=16) as h:
        J, K = torch.empty_like(Pd), torch.empty_like(Pd)
        h.build(Pd, J, K)
        torch.cuda.synchronize()
        assert quart == h.stats()["quartets_k"]                  # every quartet evaluated by exactly one rank
    assert (Js - J).abs().max().item() < 1e-11 and (Ks - K).abs().max().item() < 1e-11
    assert np.abs(Js.cpu().numpy() - ref["J"]).max() < TOL and np.abs(Ks.cpu().numpy() - ref["K"]).max() < TOL


TOL_MIXED = 1e-6


@pytest.mark.parametrize("name", ["pd_test", "water8"])
def test_mixed_precision_full_matrices(torch_cuda, oracle_mod, name):
    """Mixed-precision mode (PAPER 3.5 L817-821; north_star: <= 1e-6 Eh against the fp64 oracle, reported separately from
    the 1e-9 fp64 test): K quartets below the switch run in fp32.  A raised switch sends (nearly) all of them there."""
    from paper_2410_22278_b200 import workloads
    wl = workloads.get(name)
    P, S = _density(oracle_mod, wl)
    ref = oracle_mod.jk(wl, P)
    J, K, _, st = _gpu_jk(torch_cuda, wl, P, precision=1)
    dJ, dK = np.abs(J - ref["J"]).max(), np.abs(K - ref["K"]).max()
    print(f"mixed precision {name}: max|dJ| = {dJ:.3e}, max|dK| = {dK:.3e}, fp32 share of K quartets = "
          f"{st['quartets_k_fp32'] / max(st['quartets_k'], 1):.3f}")
    assert st["quartets_k_fp32"] > 0 and st["quartets_k_fp32"] < st["quartets_k"]
    assert dJ < TOL and dK < TOL_MIXED
    # the fp32 evaluators themselves: with the switch at 1e+3 every quartet of the classes that have a mixed kernel
    # (L <= 4) runs in fp32; errors stay those of fp32
    J2, K2, _, st2 = _gpu_jk(torch_cuda, wl, P, precision=1, mixed_switch=1e3)
    assert st2["quartets_k_fp32"] > 0.5 * st2["quartets_k"]
    dK2 = np.abs(K2 - ref["K"]).max()
    print(f"  all-fp32 quartets: max|dK| = {dK2:.3e}")
    assert dK2 < 1e-4 * max(1.0, np.abs(ref["K"]).max())


@pytest.mark.parametrize("name", ["tiny", "pd_test", "water8"])
def test_one_electron_terms(torch_cuda, oracle_mod, name):
    """kinetic matrix (SI eq S1), point-charge interaction matrix V (eq 52) and the Ewald energy of the
    charges (eq 91) against the oracle; a charged set of point charges on purpose (the -pi/(Omega w^2) terms matter)."""
    from paper_2410_22278_b200 import workloads
    from paper_2410_22278_b200.binding import PbcJK
    torch = torch_cuda
    wl = workloads.get(name)
    rng = np.random.default_rng(17)
    q = rng.uniform(0.5, 8.0, wl.natom) * rng.choice([1.0, 1.0, -1.0], wl.natom)
    ref = oracle_mod.one_electron(wl, q)
    with PbcJK(wl) as h:
        T = torch.empty((wl.nbf, wl.nbf), dtype=torch.float64, device="cuda")
        V = torch.empty_like(T)
        e = h.one_electron(q, T, V)
        torch.cuda.synchronize()
        # the J/K build still works afterwards (shared workspaces)
        P, _ = _density(oracle_mod, wl)
        Pd = torch.from_numpy(P).cuda()
        J = torch.empty_like(Pd)
        h.build(Pd, J, None)
        torch.cuda.synchronize()
        e2 = h.one_electron(q, None, None)
    T, V = T.cpu().numpy(), V.cpu().numpy()
    scale = max(1.0, np.abs(q).max())
    assert np.abs(T - ref["T"]).max() < 1e-10
    assert np.abs(V - ref["V"]).max() < TOL * scale, np.abs(V - ref["V"]).max()
    assert abs(e - ref["E_nuc"]) < 1e-9 * max(1.0, abs(ref["E_nuc"])) and abs(e2 - e) < 1e-11
    assert np.abs(T - T.T).max() < 1e-12 and np.abs(V - V.T).max() < 1e-11
    if name == "tiny":
        Jref = oracle_mod.jk(wl, P, which="j")["J"]
        assert np.abs(J.cpu().numpy() - Jref).max() < TOL


@pytest.mark.parametrize("name", ["pd_test", "water8"])
def test_orbital_entry_point(torch_cuda, oracle_mod, name):
    """pbc_jk_build_orbitals: handing C with P = C C^T gives the oracle's J and K of that P, and the same
    matrices as pbc_jk_build (which factors P itself) to rounding."""
    from paper_2410_22278_b200 import workloads
    from paper_2410_22278_b200.binding import PbcJK
    torch = torch_cuda
    wl = workloads.get(name)
    S = oracle_mod.overlap(wl)
    Cn = workloads.orthonormal_orbitals(wl.orbitals_seed(), S)
    P = Cn @ Cn.T
    ref = oracle_mod.jk(wl, 0.5 * (P + P.T))
    with PbcJK(wl) as h:
        Cd = torch.from_numpy(np.ascontiguousarray(Cn)).cuda()
        J, K, J2, K2 = (torch.empty((wl.nbf, wl.nbf), dtype=torch.float64, device="cuda") for _ in range(4))
        h.build_orbitals(Cd, J, K)
        h.build(torch.from_numpy(0.5 * (P + P.T)).cuda(), J2, K2)
        torch.cuda.synchronize()
        assert h.stats()["rank_p"] == wl.n_occ
    assert np.abs(J.cpu().numpy() - ref["J"]).max() < TOL and np.abs(K.cpu().numpy() - ref["K"]).max() < TOL
    assert (J - J2).abs().max().item() < 1e-11 and (K - K2).abs().max().item() < 1e-11


def test_entry_point_argument_errors(torch_cuda):
    """The newer entry points refuse bad arguments with a status and a message, never a crash."""
    from paper_2410_22278_b200 import workloads
    from paper_2410_22278_b200.binding import PbcJK, PbcJKError, load
    torch = torch_cuda
    wl = workloads.get("tiny")
    lib = load()
    with PbcJK(wl) as h:
        n = h.nbf
        C = torch.zeros((n, 2), dtype=torch.float64, device="cuda")
        J = torch.empty((n, n), dtype=torch.float64, device="cuda")
        assert lib.pbc_jk_build_orbitals(h._h, None, 2, J.data_ptr(), None, None) == -1
        assert lib.pbc_jk_build_orbitals(h._h, C.data_ptr(), 0, J.data_ptr(), None, None) == -1
        assert lib.pbc_jk_build_orbitals(h._h, C.data_ptr(), n + 1, J.data_ptr(), None, None) == -1
        assert b"nocc" in lib.pbc_jk_last_error(h._h)
        assert lib.pbc_jk_one_electron(h._h, None, None, J.data_ptr(), None, None) == -1
        assert lib.pbc_jk_set_shard(h._h, 2, 2) == -1 and lib.pbc_jk_set_shard(h._h, 0, 0) == -1
        assert lib.pbc_jk_set_shard(h._h, 1, 2) == 0 and lib.pbc_jk_set_shard(h._h, 0, 1) == 0
        with pytest.raises(ValueError):
            h.build_orbitals(C.float(), J)
        # a density outside the validated range of the packed lattice indices is reported, not silently mis-summed
        P = torch.eye(n, dtype=torch.float64, device="cuda") * 1e7
        h.build(P, J, None)
        with pytest.raises(PbcJKError) as ei:
            h.stats()
        assert ei.value.code == -4


def test_single_s_function_cell(torch_cuda, oracle_mod):
    """Smallest possible input: one s primitive in a cube (every list has one entry, every class but (ss|ss) is empty)."""
    from paper_2410_22278_b200 import workloads as W
    wl = W.Workload(name="one", cell=np.eye(3) * 7.0, xyz=np.array([[0.3, 0.2, 0.1]]), sh_atom=np.zeros(1, np.int32),
                    sh_l=np.zeros(1, np.int32), sh_nprim=np.ones(1, np.int32), sh_off=np.zeros(1, np.int32),
                    exps=np.array([0.9]), coefs=np.ones(1), omega=0.4, n_occ=1, seed=1)
    S = oracle_mod.overlap(wl)
    P = np.array([[1.0 / S[0, 0]]])
    ref = oracle_mod.jk(wl, P)
    J, K, Sg, st = _gpu_jk(torch_cuda, wl, P)
    assert abs(Sg[0, 0] - S[0, 0]) < 1e-13
    assert abs(J[0, 0] - ref["J"][0, 0]) < TOL and abs(K[0, 0] - ref["K"][0, 0]) < TOL
    assert abs(J[0, 0] - K[0, 0]) < TOL          # one function: (mm|mm) both ways
