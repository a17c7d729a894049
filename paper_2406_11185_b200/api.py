"""Thin ctypes binding of libadft.so (include/adft.h).  Argument marshalling only: every step of the
J/K path runs in the CUDA library.  PyTorch appears only as the owner of device memory and streams.

There is no CPU fallback: if libadft.so is missing, `lib()` raises; on a box without a GPU the compute
entry points return ADFT_ERR_CUDA.
"""
from __future__ import annotations

import ctypes as C
import os

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SO = os.path.join(_HERE, "libadft.so")
_lib = None

ADFT_COEFFS_FINAL = 0
ADFT_NORMALIZE_SHELLS = 1
ADFT_MAX_CLASSES = 120

STATUS = {0: "ADFT_OK", 1: "ADFT_ERR_INVALID_ARG", 2: "ADFT_ERR_UNSUPPORTED_L", 3: "ADFT_ERR_ALLOC",
          4: "ADFT_ERR_CUDA", 5: "ADFT_ERR_NOT_FINITE", 6: "ADFT_ERR_INTERNAL"}


class AdftError(RuntimeError):
    def __init__(self, status, msg):
        super().__init__(f"{STATUS.get(status, status)}: {msg}")
        self.status = status


class JKStats(C.Structure):
    _fields_ = [("quartets_unique", C.c_int64), ("quartets_kept", C.c_int64), ("prim_quartets", C.c_int64),
                ("prim_quartets_evaluated", C.c_int64),
                ("class_quartets", C.c_int64 * ADFT_MAX_CLASSES),
                ("class_prim_quartets", C.c_int64 * ADFT_MAX_CLASSES), ("class_ms", C.c_double * ADFT_MAX_CLASSES),
                ("class_model_flops", C.c_double * ADFT_MAX_CLASSES),
                ("model_flops", C.c_double), ("dmax", C.c_double),
                ("ms_dmax", C.c_double), ("ms_plan", C.c_double), ("ms_eri", C.c_double),
                ("ms_finalize", C.c_double), ("ms_total", C.c_double),
                ("kernel_launches", C.c_int32), ("reserved", C.c_int32),
                ("quartets_fp32", C.c_int64), ("class_quartets_fp32", C.c_int64 * ADFT_MAX_CLASSES),
                ("class_ms_fp32", C.c_double * ADFT_MAX_CLASSES)]


class JKOptions(C.Structure):
    """adft_jk_options_t (include/adft.h): flags, shard_rank, shard_count."""
    _fields_ = [("flags", C.c_uint32), ("shard_rank", C.c_int32), ("shard_count", C.c_int32), ("reserved0", C.c_int32),
                ("fp32_band", C.c_double), ("reserved", C.c_double * 3)]


ADFT_JK_BLOCK_DENSITY = 1
ADFT_JK_MIXED_PRECISION = 2

EXPORTS = ["adft_basis_nsph", "adft_cart_to_spherical", "adft_cart_to_spherical_noalloc", "adft_jk_build_ex", "adft_jk_build_incremental", "adft_basis_create", "adft_basis_nbf", "adft_basis_shell_offsets", "adft_basis_coefficients",
           "adft_shellpairs_build", "adft_shellpairs_build_ex", "adft_shellpairs_prim_counts", "adft_shellpairs_schwarz", "adft_jk_build", "adft_jk_build_host", "adft_jk_stats",
           "adft_shellpairs_counts", "adft_shellpairs_destroy", "adft_basis_destroy", "adft_status_string",
           "adft_last_error", "adft_fp64_peak_tflops"]


def lib():
    global _lib
    if _lib is None:
        if not os.path.exists(_SO):
            raise ImportError(f"{_SO} is missing: run `python -m paper_2406_11185_b200.build` "
                              "(the J/K path has no CPU fallback)")
        L = C.CDLL(_SO)
        L.adft_status_string.restype = C.c_char_p
        L.adft_last_error.restype = C.c_char_p
        L.adft_shellpairs_destroy.restype = None
        L.adft_basis_destroy.restype = None
        L.adft_jk_build.argtypes = [C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p, C.c_double, C.c_void_p]
        L.adft_jk_build_ex.argtypes = [C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p, C.c_double, C.c_void_p, C.c_void_p]
        L.adft_jk_build_incremental.argtypes = [C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p, C.c_double,
                                                C.c_void_p, C.c_void_p]
        L.adft_cart_to_spherical.argtypes = [C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p]
        L.adft_cart_to_spherical_noalloc.argtypes = [C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p]
        L.adft_jk_build_host.argtypes = [C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p, C.c_double, C.c_void_p]
        L.adft_shellpairs_build.argtypes = [C.c_void_p, C.c_void_p, C.c_void_p]
        L.adft_shellpairs_build_ex.argtypes = [C.c_void_p, C.c_double, C.c_void_p, C.c_void_p]
        L.adft_jk_stats.argtypes = [C.c_void_p, C.c_void_p]
        L.adft_fp64_peak_tflops.argtypes = [C.c_void_p, C.c_void_p]
        _lib = L
    return _lib


def _check(rc):
    if rc != 0:
        raise AdftError(rc, lib().adft_last_error().decode())


def _stream_ptr(stream):
    if stream is None:
        import torch
        return C.c_void_p(torch.cuda.current_stream().cuda_stream)
    if hasattr(stream, "cuda_stream"):
        return C.c_void_p(stream.cuda_stream)
    return C.c_void_p(int(stream))


class Basis:
    """adft_basis_create: host arrays in, opaque handle out."""

    def __init__(self, atoms, shells, exponents, coefficients, normalize=True):
        self._h = C.c_void_p()
        atoms = np.ascontiguousarray(atoms, np.float64)
        shells = np.ascontiguousarray(shells, np.int32)        # [nshells,4] {atom,l,nprim,prim_offset}
        e = np.ascontiguousarray(exponents, np.float64)
        c = np.ascontiguousarray(coefficients, np.float64)
        _check(lib().adft_basis_create(C.c_int32(atoms.shape[0]), atoms.ctypes.data_as(C.c_void_p),
                                       C.c_int32(shells.shape[0]), shells.ctypes.data_as(C.c_void_p),
                                       e.ctypes.data_as(C.c_void_p), c.ctypes.data_as(C.c_void_p),
                                       C.c_uint32(ADFT_NORMALIZE_SHELLS if normalize else ADFT_COEFFS_FINAL),
                                       C.byref(self._h)))
        n = C.c_int32()
        _check(lib().adft_basis_nbf(self._h, C.byref(n)))
        self.nbf = int(n.value)
        self.nshells = int(shells.shape[0])
        self.nprim = int(e.shape[0])

    @classmethod
    def from_workload(cls, w, normalize=True):
        return cls(w.atoms, w.shells_struct(), w.exponents, w.coefficients, normalize=normalize)

    def shell_offsets(self):
        out = np.zeros(self.nshells + 1, np.int32)
        _check(lib().adft_basis_shell_offsets(self._h, out.ctypes.data_as(C.c_void_p)))
        return out

    def coefficients(self):
        out = np.zeros(self.nprim, np.float64)
        _check(lib().adft_basis_coefficients(self._h, out.ctypes.data_as(C.c_void_p)))
        return out

    def close(self):
        if self._h:
            lib().adft_basis_destroy(self._h)
            self._h = C.c_void_p()

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass


class ShellPairs:
    """adft_shellpairs_build + adft_jk_build on torch CUDA tensors."""

    def __init__(self, basis: Basis, stream=None, prim_threshold=None):
        self.basis = basis
        self._h = C.c_void_p()
        if prim_threshold is None:
            _check(lib().adft_shellpairs_build(basis._h, _stream_ptr(stream), C.byref(self._h)))
        else:
            _check(lib().adft_shellpairs_build_ex(basis._h, C.c_double(prim_threshold), _stream_ptr(stream),
                                                  C.byref(self._h)))

    def prim_counts(self):
        a, b, t = C.c_int64(), C.c_int64(), C.c_double()
        _check(lib().adft_shellpairs_prim_counts(self._h, C.byref(a), C.byref(b), C.byref(t)))
        return int(a.value), int(b.value), float(t.value)

    def schwarz(self):
        Q = np.zeros((self.basis.nshells, self.basis.nshells), np.float64)
        _check(lib().adft_shellpairs_schwarz(self._h, Q.ctypes.data_as(C.c_void_p)))
        return Q

    def counts(self):
        a, b = C.c_int64(), C.c_int64()
        _check(lib().adft_shellpairs_counts(self._h, C.byref(a), C.byref(b)))
        return int(a.value), int(b.value)

    def _check_tensors(self, *ts):
        N = self.basis.nbf
        for t in ts:
            if t is not None:
                assert t.is_cuda and t.dtype.is_floating_point and t.element_size() == 8 and t.is_contiguous()
                assert tuple(t.shape) == (N, N)

    @staticmethod
    def _options(block_density, shard, mixed_precision=False, fp32_band=0.0):
        o = JKOptions()
        o.flags = (ADFT_JK_BLOCK_DENSITY if block_density else 0) | (ADFT_JK_MIXED_PRECISION if mixed_precision else 0)
        o.fp32_band = float(fp32_band)
        if shard is not None:
            o.shard_rank, o.shard_count = int(shard[0]), int(shard[1])
        return o

    def jk_build(self, D, J=None, K=None, tau=0.0, stream=None, block_density=False, shard=None, mixed_precision=False,
                 fp32_band=0.0):
        """D, J, K: torch.float64 CUDA tensors [N,N] (J or K may be None).  Enqueues on `stream`.
        block_density: the screen of DESIGN.md R-23; shard = (rank, count): only this rank's share of the tiles
        (partial J, K; see jk_build_distributed); mixed_precision: quartets with tau <= S < fp32_band*tau (default 1e5)
        in single precision."""
        self._check_tensors(D, J, K)
        if not block_density and shard is None and not mixed_precision:
            _check(lib().adft_jk_build(self._h, C.c_void_p(D.data_ptr()),
                                       C.c_void_p(J.data_ptr()) if J is not None else None,
                                       C.c_void_p(K.data_ptr()) if K is not None else None,
                                       C.c_double(tau), _stream_ptr(stream)))
            return
        o = self._options(block_density, shard, mixed_precision, fp32_band)
        _check(lib().adft_jk_build_ex(self._h, C.c_void_p(D.data_ptr()),
                                      C.c_void_p(J.data_ptr()) if J is not None else None,
                                      C.c_void_p(K.data_ptr()) if K is not None else None,
                                      C.c_double(tau), C.byref(o), _stream_ptr(stream)))

    def jk_build_incremental(self, D, D_prev, J=None, K=None, tau=0.0, stream=None, shard=None):
        """adft_jk_build_incremental: J, K hold the matrices of D_prev on entry and those of D on exit; D_prev <- D."""
        self._check_tensors(D, D_prev, J, K)
        o = self._options(True, shard)
        _check(lib().adft_jk_build_incremental(self._h, C.c_void_p(D.data_ptr()), C.c_void_p(D_prev.data_ptr()),
                                               C.c_void_p(J.data_ptr()) if J is not None else None,
                                               C.c_void_p(K.data_ptr()) if K is not None else None,
                                               C.c_double(tau), C.byref(o), _stream_ptr(stream)))

    def jk_build_distributed(self, D, J=None, K=None, tau=0.0, group=None, block_density=False):
        """Sharded build over the ranks of a torch.distributed process group (PAPER.md:105, 283-291:
        replicated D, independent quartet batches, one reduction): every rank holds the same D and pair table, evaluates
        the tiles t with t % world == rank, and the partial J, K are summed with one all-reduce each (NCCL over
        NVLink on GPUs).  On return every rank holds the full J and K."""
        rank, world = shard_of(group)
        self.jk_build(D, J, K, tau, block_density=block_density, shard=(rank, world) if world > 1 else None)
        allreduce_jk(J, K, group)

    def jk_build_host(self, D, J=None, K=None, tau=0.0, stream=None):
        """D, J, K: numpy float64 [N,N] host arrays (pinned or not); copies are inside the call."""
        _check(lib().adft_jk_build_host(self._h, C.c_void_p(D.ctypes.data),
                                        C.c_void_p(J.ctypes.data) if J is not None else None,
                                        C.c_void_p(K.ctypes.data) if K is not None else None,
                                        C.c_double(tau), _stream_ptr(stream)))

    def cart_to_spherical(self, M, out=None, stream=None):
        """adft_cart_to_spherical: M [N,N] (J or K) -> [nsph,nsph] in real solid harmonics, m = -l..l inside a shell."""
        import torch
        self._check_tensors(M)
        n = C.c_int32()
        _check(lib().adft_basis_nsph(self.basis._h, C.byref(n)))
        if out is None:
            out = torch.empty(n.value, n.value, dtype=torch.float64, device=M.device)
        assert out.is_cuda and out.is_contiguous() and tuple(out.shape) == (n.value, n.value) and out.element_size() == 8
        _check(lib().adft_cart_to_spherical(self._h, C.c_void_p(M.data_ptr()), C.c_void_p(out.data_ptr()), _stream_ptr(stream)))
        return out

    def cart_to_spherical_noalloc(self, M, out, stream=None):
        """adft_cart_to_spherical_noalloc (include/adft_noalloc.h): the same transform with its working memory in the
        library's static device array: no allocation here or in the library, so the caller passes `out` [nsph,nsph]."""
        self._check_tensors(M)
        n = C.c_int32()
        _check(lib().adft_basis_nsph(self.basis._h, C.byref(n)))
        assert out.is_cuda and out.is_contiguous() and out.element_size() == 8 and tuple(out.shape) == (n.value, n.value)
        _check(lib().adft_cart_to_spherical_noalloc(self._h, C.c_void_p(M.data_ptr()), C.c_void_p(out.data_ptr()), _stream_ptr(stream)))
        return out

    def stats(self) -> JKStats:
        s = JKStats()
        _check(lib().adft_jk_stats(self._h, C.byref(s)))
        return s

    def close(self):
        if self._h:
            lib().adft_shellpairs_destroy(self._h)
            self._h = C.c_void_p()

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass


def shard_of(group=None):
    """(rank, world size) of this process in `group`; (0, 1) when torch.distributed is not initialised."""
    import torch.distributed as dist
    if not (dist.is_available() and dist.is_initialized()):
        return 0, 1
    return dist.get_rank(group), dist.get_world_size(group)


def allreduce_jk(J, K, group=None):
    """The one exchange step of the sharded build: sum the ranks' partial J and K in place (no-op for one rank)."""
    import torch.distributed as dist
    if not (dist.is_available() and dist.is_initialized()) or dist.get_world_size(group) == 1:
        return
    for M in (J, K):
        if M is not None:
            dist.all_reduce(M, op=dist.ReduceOp.SUM, group=group)


def fp64_peak_tflops(stream=None) -> float:
    v = C.c_double()
    _check(lib().adft_fp64_peak_tflops(_stream_ptr(stream), C.byref(v)))
    return float(v.value)


def jk(workload, tau=None, want_j=True, want_k=True, prim_threshold=None, block_density=False, D=None,
       mixed_precision=False, fp32_band=0.0):
    """Convenience: full path on cuda:0 for a workloads.Workload; returns numpy J, K and the stats."""
    import torch
    bs = Basis.from_workload(workload)
    sp = ShellPairs(bs, prim_threshold=prim_threshold)
    D = torch.from_numpy(np.ascontiguousarray(workload.D if D is None else D)).cuda()
    J = torch.empty_like(D) if want_j else None
    K = torch.empty_like(D) if want_k else None
    sp.jk_build(D, J, K, workload.tau if tau is None else tau, block_density=block_density,
                mixed_precision=mixed_precision, fp32_band=fp32_band)
    torch.cuda.synchronize()
    st = sp.stats()
    out = (J.cpu().numpy() if want_j else None, K.cpu().numpy() if want_k else None, st, sp.schwarz())
    sp.close(); bs.close()
    return out
