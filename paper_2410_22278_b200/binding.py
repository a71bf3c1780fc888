"""Thin ctypes binding of libpbc_jk.so (include/pbc_jk.h).  Argument marshalling only: every step
of the path runs in the CUDA kernels behind the C ABI.  PyTorch supplies device memory and streams.

There is no fallback: if the shared library is missing or no CUDA device is present the calls
raise.
"""
from __future__ import annotations

import ctypes as C
import os
from typing import Optional

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libpbc_jk.so")

PBC_JK_OK = 0
STATUS = {0: "OK", -1: "INVALID_ARG", -2: "NOMEM", -3: "CUDA", -4: "UNSUPPORTED"}

# every symbol include/pbc_jk.h declares (checked by tests/test_abi.py)
SYMBOLS = ["pbc_jk_create", "pbc_jk_nbf", "pbc_jk_overlap", "pbc_jk_overlap_noalloc", "pbc_jk_build", "pbc_jk_build_orbitals", "pbc_jk_build_host",
           "pbc_jk_one_electron", "pbc_jk_set_parts", "pbc_jk_set_shard", "pbc_jk_get_stats", "pbc_jk_set_profile", "pbc_jk_get_class_stats",
           "pbc_jk_last_error", "pbc_jk_destroy"]


class pbc_cell(C.Structure):
    _fields_ = [("a", C.c_double * 9)]


class pbc_atoms(C.Structure):
    _fields_ = [("natom", C.c_int32), ("xyz", C.POINTER(C.c_double))]


class pbc_shells(C.Structure):
    _fields_ = [("nshell", C.c_int32), ("atom", C.POINTER(C.c_int32)), ("l", C.POINTER(C.c_int32)),
                ("nprim", C.POINTER(C.c_int32)), ("prim_off", C.POINTER(C.c_int32)),
                ("exps", C.POINTER(C.c_double)), ("coefs", C.POINTER(C.c_double))]


class pbc_cutoffs(C.Structure):
    _fields_ = [("r_cut", C.c_double), ("g_cut", C.c_double), ("d_pair", C.c_double), ("d_schwarz", C.c_double),
                ("d_ewald_k", C.c_double), ("precision", C.c_int32), ("mixed_switch", C.c_double),
                ("lr_g_batch", C.c_int32), ("g_min", C.c_double)]


class pbc_jk_stats_t(C.Structure):
    _fields_ = [("nbf", C.c_int32), ("nshell", C.c_int32), ("natom", C.c_int32), ("n_g", C.c_int32),
                ("n_prim_pairs", C.c_int64), ("n_shell_pair_images", C.c_int64),
                ("quartets_j", C.c_int64), ("quartets_k", C.c_int64),
                ("candidates_j", C.c_int64), ("candidates_k", C.c_int64),
                ("ms_density", C.c_double), ("ms_sr_j", C.c_double), ("ms_sr_k", C.c_double), ("ms_lr", C.c_double),
                ("ms_total", C.c_double), ("create_seconds", C.c_double), ("n_launches", C.c_int64),
                ("quartets_k_fp32", C.c_int64), ("ms_lr_gemm", C.c_double), ("rank_p", C.c_int32)]


class pbc_jk_class_stat(C.Structure):
    _fields_ = [("kind", C.c_int32), ("l", C.c_int32 * 4), ("quartets", C.c_int64), ("candidates", C.c_int64),
                ("ms", C.c_double)]


_lib = None


def load() -> C.CDLL:
    """dlopen libpbc_jk.so (built by `python -m paper_2410_22278_b200.build`).  Raises if absent."""
    global _lib
    if _lib is None:
        if not os.path.exists(LIB_PATH):
            raise RuntimeError(f"{LIB_PATH} is missing: build it with `python -m paper_2410_22278_b200.build` "
                               "(there is no CPU fallback)")
        lib = C.CDLL(LIB_PATH)
        lib.pbc_jk_create.argtypes = [C.POINTER(pbc_cell), C.POINTER(pbc_atoms), C.POINTER(pbc_shells), C.c_double,
                                      C.POINTER(pbc_cutoffs), C.POINTER(C.c_void_p)]
        lib.pbc_jk_create.restype = C.c_int
        lib.pbc_jk_nbf.argtypes = [C.c_void_p]
        lib.pbc_jk_nbf.restype = C.c_int
        lib.pbc_jk_overlap.argtypes = [C.c_void_p, C.c_void_p]
        lib.pbc_jk_overlap.restype = C.c_int
        lib.pbc_jk_overlap_noalloc.argtypes = [C.c_void_p, C.c_void_p, C.c_void_p]
        lib.pbc_jk_overlap_noalloc.restype = C.c_int
        lib.pbc_jk_build.argtypes = [C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p]
        lib.pbc_jk_build.restype = C.c_int
        lib.pbc_jk_build_orbitals.argtypes = [C.c_void_p, C.c_void_p, C.c_int32, C.c_void_p, C.c_void_p, C.c_void_p]
        lib.pbc_jk_build_orbitals.restype = C.c_int
        lib.pbc_jk_build_host.argtypes = [C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p]
        lib.pbc_jk_build_host.restype = C.c_int
        lib.pbc_jk_set_parts.argtypes = [C.c_void_p, C.c_int32]
        lib.pbc_jk_set_parts.restype = C.c_int
        lib.pbc_jk_get_stats.argtypes = [C.c_void_p, C.POINTER(pbc_jk_stats_t)]
        lib.pbc_jk_get_stats.restype = C.c_int
        lib.pbc_jk_set_profile.argtypes = [C.c_void_p, C.c_int32]
        lib.pbc_jk_set_profile.restype = C.c_int
        lib.pbc_jk_get_class_stats.argtypes = [C.c_void_p, C.POINTER(pbc_jk_class_stat), C.c_int32,
                                               C.POINTER(C.c_int32)]
        lib.pbc_jk_get_class_stats.restype = C.c_int
        lib.pbc_jk_last_error.argtypes = [C.c_void_p]
        lib.pbc_jk_last_error.restype = C.c_char_p
        lib.pbc_jk_destroy.argtypes = [C.c_void_p]
        lib.pbc_jk_destroy.restype = C.c_int
        lib.pbc_jk_one_electron.argtypes = [C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p, C.POINTER(C.c_double), C.c_void_p]
        lib.pbc_jk_one_electron.restype = C.c_int
        lib.pbc_jk_set_shard.argtypes = [C.c_void_p, C.c_int32, C.c_int32]
        lib.pbc_jk_set_shard.restype = C.c_int
        _lib = lib
    return _lib


class PbcJKError(RuntimeError):
    def __init__(self, code: int, text: str):
        super().__init__(f"pbc_jk: {STATUS.get(code, code)}: {text}")
        self.code = code


def _dp(a):
    return a.ctypes.data_as(C.POINTER(C.c_double))


def _ip(a):
    return a.ctypes.data_as(C.POINTER(C.c_int32))


_PARTS = {"sr": 1, "lr": 2, "self": 4}


def allreduce_jk(J, K, group=None):
    """The one collective of the sharded build: sum the ranks' partial J and K in place.  One message when J and K
    sit back to back in memory (allocate them as two halves of one buffer), else one staging copy."""
    import torch
    import torch.distributed as dist

    parts = [t for t in (J, K) if t is not None]
    if not parts or not dist.is_initialized() or dist.get_world_size(group) == 1:
        return
    if len(parts) == 2 and J.is_contiguous() and K.is_contiguous() and \
            J.data_ptr() + J.numel() * J.element_size() == K.data_ptr() and J.untyped_storage().data_ptr() == K.untyped_storage().data_ptr():
        both = torch.as_strided(J, (J.numel() + K.numel(),), (1,))
        dist.all_reduce(both, group=group)
        return
    buf = torch.cat([t.reshape(-1) for t in parts])
    dist.all_reduce(buf, group=group)
    o = 0
    for t in parts:
        t.copy_(buf[o:o + t.numel()].view_as(t))
        o += t.numel()


class PbcJK:
    """One geometry: pbc_jk_create ... pbc_jk_destroy.  `wl` is a workloads.Workload (or anything
    with the same fields)."""

    def __init__(self, wl, omega: Optional[float] = None, r_cut: Optional[float] = None,
                 g_cut: Optional[float] = None, d_pair: float = 0.0, d_schwarz: Optional[float] = None,
                 d_ewald_k: float = 0.0, precision: int = 0, mixed_switch: float = 0.0, lr_g_batch: int = 0,
                 g_min: float = 0.0):
        self._h = C.c_void_p()
        lib = load()
        cell = pbc_cell()
        flat = np.ascontiguousarray(wl.cell, dtype=np.float64).ravel()
        for i in range(9):
            cell.a[i] = float(flat[i])
        self._keep = dict(
            xyz=np.ascontiguousarray(wl.xyz, dtype=np.float64), atom=np.ascontiguousarray(wl.sh_atom, dtype=np.int32),
            l=np.ascontiguousarray(wl.sh_l, dtype=np.int32), nprim=np.ascontiguousarray(wl.sh_nprim, dtype=np.int32),
            off=np.ascontiguousarray(wl.sh_off, dtype=np.int32), exps=np.ascontiguousarray(wl.exps, dtype=np.float64),
            coefs=np.ascontiguousarray(wl.coefs, dtype=np.float64))
        k = self._keep
        atoms = pbc_atoms(int(k["xyz"].shape[0]), _dp(k["xyz"]))
        shells = pbc_shells(int(k["l"].shape[0]), _ip(k["atom"]), _ip(k["l"]), _ip(k["nprim"]), _ip(k["off"]),
                            _dp(k["exps"]), _dp(k["coefs"]))
        cut = pbc_cutoffs()
        cut.r_cut = float(getattr(wl, "r_cut", 0.0) if r_cut is None else r_cut)
        cut.g_cut = float(getattr(wl, "g_cut", 0.0) if g_cut is None else g_cut)
        cut.d_pair = float(d_pair)
        cut.d_schwarz = float(getattr(wl, "tau_schwarz", 0.0) if d_schwarz is None else d_schwarz)
        cut.d_ewald_k = float(d_ewald_k)
        cut.precision = int(precision)
        cut.mixed_switch = float(mixed_switch)
        cut.lr_g_batch = int(lr_g_batch)
        cut.g_min = float(g_min)
        om = float(wl.omega if omega is None else omega)
        rc = lib.pbc_jk_create(C.byref(cell), C.byref(atoms), C.byref(shells), om, C.byref(cut), C.byref(self._h))
        if rc != PBC_JK_OK:
            raise PbcJKError(rc, (lib.pbc_jk_last_error(None) or b"").decode())
        self.nbf = int(lib.pbc_jk_nbf(self._h))

    def _check(self, rc: int):
        if rc != PBC_JK_OK:
            raise PbcJKError(rc, (load().pbc_jk_last_error(self._h) or b"").decode())

    def overlap(self) -> np.ndarray:
        S = np.zeros((self.nbf, self.nbf))
        self._check(load().pbc_jk_overlap(self._h, S.ctypes.data))
        return S

    def overlap_noalloc(self, S_dev, stream=None):
        """S into a caller's device tensor (N x N fp64, overwritten) through the entry point that allocates nothing: its
        scratch is a static device array inside the library (N padded to 64 must not exceed PBC_JK_NOALLOC_MAX_NBF = 512).
        Every call shares that array: calls that overlap on the GPU race."""
        import torch

        n = self.nbf
        if not (S_dev.is_cuda and S_dev.dtype == torch.float64 and S_dev.is_contiguous() and tuple(S_dev.shape) == (n, n)):
            raise ValueError("S_dev must be a contiguous float64 CUDA tensor of shape (nbf, nbf)")
        st = torch.cuda.current_stream().cuda_stream if stream is None else int(stream)
        self._check(load().pbc_jk_overlap_noalloc(self._h, S_dev.data_ptr(), st))
        return S_dev

    def set_parts(self, parts: str = "sr+lr+self"):
        m = 0
        for p in parts.split("+"):
            m |= _PARTS[p.strip()]
        self._check(load().pbc_jk_set_parts(self._h, m))

    def one_electron(self, charges, T=None, V=None, want_e_nuc: bool = True, stream=None):
        """Kinetic matrix T, point-charge interaction matrix V (device tensors, overwritten) and the Ewald energy of the
        charges (returned; None unless want_e_nuc).  charges: one per atom (host)."""
        import torch

        n = self.nbf
        for t in (T, V):
            if t is not None and not (t.is_cuda and t.dtype == torch.float64 and t.is_contiguous() and tuple(t.shape) == (n, n)):
                raise ValueError("T, V must be contiguous float64 CUDA tensors of shape (nbf, nbf)")
        q = np.ascontiguousarray(charges, dtype=np.float64)
        assert q.shape == (self._keep["xyz"].shape[0],)
        e = C.c_double()
        st = torch.cuda.current_stream().cuda_stream if stream is None else int(stream)
        self._check(load().pbc_jk_one_electron(self._h, q.ctypes.data, T.data_ptr() if T is not None else None,
                                               V.data_ptr() if V is not None else None, C.byref(e) if want_e_nuc else None, st))
        return float(e.value) if want_e_nuc else None

    def set_shard(self, rank: int = 0, nranks: int = 1):
        """This handle builds share `rank` of `nranks` of every J and K; the sum over ranks is the full matrix."""
        self._check(load().pbc_jk_set_shard(self._h, int(rank), int(nranks)))
        self._shard = (int(rank), int(nranks))

    def build_sharded(self, P, J=None, K=None, group=None):
        """Multi-GPU build: every rank of `group` holds a handle of the same geometry with
        set_shard(rank, world) and calls this with the same P; the partial matrices are summed with ONE
        all-reduce of [J; K] over torch.distributed (NCCL over NVLink on GPUs)."""
        self.build(P, J, K)
        allreduce_jk(J, K, group)

    def build(self, P, J=None, K=None, stream=None):
        """Device tensors (torch, float64, contiguous N x N).  Enqueues on `stream` (default: torch's
        current stream) and returns without synchronising."""
        import torch

        n = self.nbf
        for t in (P, J, K):
            if t is None:
                continue
            if not (t.is_cuda and t.dtype == torch.float64 and t.is_contiguous() and tuple(t.shape) == (n, n)):
                raise ValueError("P, J, K must be contiguous float64 CUDA tensors of shape (nbf, nbf)")
        st = torch.cuda.current_stream().cuda_stream if stream is None else int(stream)
        self._check(load().pbc_jk_build(self._h, P.data_ptr(), J.data_ptr() if J is not None else None,
                                        K.data_ptr() if K is not None else None, st))

    def build_orbitals(self, Corb, J=None, K=None, stream=None):
        """Occupied-orbital entry point: Corb is a contiguous float64 CUDA tensor (nbf, nocc), P = Corb Corb^T."""
        import torch

        n = self.nbf
        if not (Corb.is_cuda and Corb.dtype == torch.float64 and Corb.is_contiguous() and Corb.dim() == 2 and Corb.shape[0] == n):
            raise ValueError("Corb must be a contiguous float64 CUDA tensor of shape (nbf, nocc)")
        for t in (J, K):
            if t is not None and not (t.is_cuda and t.dtype == torch.float64 and t.is_contiguous() and tuple(t.shape) == (n, n)):
                raise ValueError("J, K must be contiguous float64 CUDA tensors of shape (nbf, nbf)")
        st = torch.cuda.current_stream().cuda_stream if stream is None else int(stream)
        self._check(load().pbc_jk_build_orbitals(self._h, Corb.data_ptr(), int(Corb.shape[1]), J.data_ptr() if J is not None else None,
                                                 K.data_ptr() if K is not None else None, st))

    def build_host(self, P: np.ndarray, want_j: bool = True, want_k: bool = True):
        """Host numpy in, host numpy out (copies inside the library); synchronous."""
        n = self.nbf
        P = np.ascontiguousarray(P, dtype=np.float64)
        assert P.shape == (n, n)
        J = np.empty((n, n)) if want_j else None
        K = np.empty((n, n)) if want_k else None
        self._check(load().pbc_jk_build_host(self._h, P.ctypes.data, J.ctypes.data if want_j else None,
                                             K.ctypes.data if want_k else None))
        return J, K

    def build_host_ptr(self, p_ptr: int, j_ptr: int, k_ptr: int):
        """Same with raw host addresses (pinned torch tensors in bench.py)."""
        self._check(load().pbc_jk_build_host(self._h, p_ptr, j_ptr or None, k_ptr or None))

    def stats(self) -> dict:
        s = pbc_jk_stats_t()
        self._check(load().pbc_jk_get_stats(self._h, C.byref(s)))
        return {f: getattr(s, f) for f, _ in s._fields_}

    def set_profile(self, on: bool = True):
        self._check(load().pbc_jk_set_profile(self._h, 1 if on else 0))

    def class_stats(self) -> list:
        """Per real-space kernel class of the last build: kind ('J'|'K'), l, quartets, candidates, ms."""
        cap = 128
        arr = (pbc_jk_class_stat * cap)()
        n = C.c_int32()
        self._check(load().pbc_jk_get_class_stats(self._h, arr, cap, C.byref(n)))
        out = []
        for i in range(min(n.value, cap)):
            s = arr[i]
            nl = 2 if s.kind == 0 else 4
            out.append(dict(kind="J" if s.kind == 0 else "K", l=tuple(int(s.l[k]) for k in range(nl)),
                            quartets=int(s.quartets), candidates=int(s.candidates), ms=float(s.ms)))
        return out

    def close(self):
        if self._h:
            load().pbc_jk_destroy(self._h)
            self._h = C.c_void_p()

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def __enter__(self):
        return self

    def __exit__(self, *a):
        self.close()


PEAKS_LIB_PATH = os.path.join(_HERE, "libpbc_jk_benchpeaks.so")


def bench_peaks(iters: int = 20000) -> dict:
    """bench.py's roofline denominators measured on the current device (helper library outside the product ABI):
    FP64 FMA, FP32 FMA and FP64 tensor-core (DMMA) TFLOP/s; `fp64_mixed_pipe` = DMMA and DFMA warps side by side (sum of
    both rates: equal to the single peaks when the two share a pipe), `fp64_dmma_loop` = the GEMM's inner loop (shared-memory
    fragment loads + DMMA + barrier) without its global loads."""
    if not os.path.exists(PEAKS_LIB_PATH):
        raise RuntimeError(f"{PEAKS_LIB_PATH} is missing: build it with `python -m paper_2410_22278_b200.build`")
    lib = C.CDLL(PEAKS_LIB_PATH)
    out = {}
    for name in ("fp64_fma", "fp32_fma", "fp64_dmma", "fp64_mixed_pipe", "fp64_dmma_loop"):
        f = getattr(lib, f"bench_{name}_peak")
        f.argtypes = [C.c_int32, C.POINTER(C.c_double)]
        f.restype = C.c_int
        v = C.c_double()
        if f(int(iters), C.byref(v)) != 0:
            raise RuntimeError(f"bench_{name}_peak failed (no CUDA device?)")
        out[name] = float(v.value)
    return out
