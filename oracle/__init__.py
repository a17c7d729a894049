"""ORACLE -- TEST INFRASTRUCTURE ONLY (see oracle/jk_oracle.c header).

ctypes binding of the plain C fp64 oracle.  Only tests/, __graft_entry__.smoke() and bench.py's
cpu_baseline / --impl reference legs may import this package.  It imports nothing from the product
package except nothing at all: inputs arrive as plain numpy arrays.
"""
from __future__ import annotations

import ctypes as C
import os
import subprocess
import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SO = os.path.join(_HERE, "liboracle.so")
_SO_G = os.path.join(_HERE, "liboracle_g.so")      # the same source with -DLMAX_SHELL=4 (g shells)
_SRC = [os.path.join(_HERE, "jk_oracle.c"), os.path.join(_HERE, "eri_core.inc.c")]
_lib = None
_lib_g = None
NQCLASS = 120          # quartet classes up to g; the l <= 3 classes keep their indices 0..54


def _compile(so, extra, force):
    if not force and os.path.exists(so) and all(os.path.getmtime(so) >= os.path.getmtime(s) for s in _SRC):
        return so
    cmd = ["gcc", "-O2", "-std=c11", "-fopenmp", "-fPIC", "-shared", *extra, "-o", so, _SRC[0], "-lm"]
    subprocess.run(cmd, check=True, cwd=_HERE)
    return so


def build(force: bool = False) -> str:
    """Compile oracle/liboracle.so (l <= 3) and oracle/liboracle_g.so (l <= 4) with gcc (plain C, -O2, OpenMP, no
    fast-math).  Two builds of one source: the table strides of the integral core grow with the highest l, and the
    hours-long l <= 3 runs should not pay for g."""
    _compile(_SO_G, ["-DLMAX_SHELL=4"], force)
    return _compile(_SO, [], force)


def lib(lmax: int = 3):
    """The oracle library for shells up to lmax (3: liboracle.so; 4: liboracle_g.so)."""
    global _lib, _lib_g
    if lmax <= 3:
        if _lib is None:
            build()
            _lib = C.CDLL(_SO)
            _lib.orc_dmax.restype = C.c_double
        return _lib
    if _lib_g is None:
        build()
        _lib_g = C.CDLL(_SO_G)
        _lib_g.orc_dmax.restype = C.c_double
        assert _lib_g.orc_lmax() == 4
    return _lib_g


def _counts_out(nq_lib_array):
    """Per-class counts as a length-NQCLASS array whichever library wrote them."""
    out = np.zeros(NQCLASS, dtype=np.int64)
    out[:len(nq_lib_array)] = nq_lib_array
    return out


def _p(a, t):
    return a.ctypes.data_as(C.POINTER(t))


class Basis:
    """Plain container of the arrays the C oracle takes (FINAL coefficients)."""

    def __init__(self, atoms, shell_atom, shell_l, shell_nprim, shell_off, exponents, coefficients):
        self.xyz = np.ascontiguousarray(atoms, dtype=np.float64)
        self.atom = np.ascontiguousarray(shell_atom, dtype=np.int32)
        self.l = np.ascontiguousarray(shell_l, dtype=np.int32)
        self.nprim = np.ascontiguousarray(shell_nprim, dtype=np.int32)
        self.off = np.ascontiguousarray(shell_off, dtype=np.int32)
        self.expo = np.ascontiguousarray(exponents, dtype=np.float64)
        self.coef = np.ascontiguousarray(coefficients, dtype=np.float64)
        self.nshells = int(self.l.shape[0])
        self.natoms = int(self.xyz.shape[0])
        self.lmax = int(self.l.max())
        self.ncart = [(int(x) + 1) * (int(x) + 2) // 2 for x in self.l]
        self.bf_off = np.concatenate([[0], np.cumsum(self.ncart)]).astype(np.int64)
        self.nbf = int(self.bf_off[-1])

    def args(self):
        return (C.c_int(self.natoms), _p(self.xyz, C.c_double), C.c_int(self.nshells), _p(self.atom, C.c_int32),
                _p(self.l, C.c_int32), _p(self.nprim, C.c_int32), _p(self.off, C.c_int32),
                _p(self.expo, C.c_double), _p(self.coef, C.c_double))


def normalize(shell_l, shell_nprim, shell_off, exponents, coef_raw):
    """SURVEY R-1 normalisation: raw contraction coefficients -> final d_k."""
    l = np.ascontiguousarray(shell_l, np.int32); n = np.ascontiguousarray(shell_nprim, np.int32)
    o = np.ascontiguousarray(shell_off, np.int32)
    e = np.ascontiguousarray(exponents, np.float64); c = np.ascontiguousarray(coef_raw, np.float64)
    out = np.empty_like(c)
    rc = lib(int(l.max())).orc_normalize(C.c_int(len(l)), _p(l, C.c_int32), _p(n, C.c_int32), _p(o, C.c_int32),
                             _p(e, C.c_double), _p(c, C.c_double), _p(out, C.c_double))
    if rc:
        raise ValueError(f"orc_normalize rc={rc}")
    return out


def basis_from_workload(w, normalize_shells=True) -> Basis:
    coef = normalize(w.shell_l, w.shell_nprim, w.shell_off, w.exponents, w.coefficients) if normalize_shells \
        else w.coefficients
    return Basis(w.atoms, w.shell_atom, w.shell_l, w.shell_nprim, w.shell_off, w.exponents, coef)


def boys(mmax: int, T: float) -> np.ndarray:
    F = np.zeros(mmax + 1, dtype=np.float64)
    lib().orc_boys(C.c_int(mmax), C.c_double(T), _p(F, C.c_double))
    return F


def boys_ld(mmax: int, T: float) -> np.ndarray:
    F = np.zeros(mmax + 1, dtype=np.longdouble)
    lib().orc_boys_ld(C.c_int(mmax), C.c_longdouble(T), _p(F, C.c_longdouble))
    return F


def eri_block(bs: Basis, A, B, Cc, D, long_double=False) -> np.ndarray:
    shape = (bs.ncart[A], bs.ncart[B], bs.ncart[Cc], bs.ncart[D])
    if long_double:
        out = np.zeros(shape, dtype=np.longdouble)
        rc = lib(bs.lmax).orc_eri_block_ld(*bs.args(), C.c_int(A), C.c_int(B), C.c_int(Cc), C.c_int(D),
                                    _p(out, C.c_longdouble))
    else:
        out = np.zeros(shape, dtype=np.float64)
        rc = lib(bs.lmax).orc_eri_block(*bs.args(), C.c_int(A), C.c_int(B), C.c_int(Cc), C.c_int(D), _p(out, C.c_double))
    if rc:
        raise ValueError(f"orc_eri_block rc={rc}")
    return out


def eri_tensor(bs: Basis) -> np.ndarray:
    """All N^4 integrals (tiny systems only), every ordered shell quartet computed on its own."""
    N = bs.nbf
    G = np.zeros((N, N, N, N))
    o = bs.bf_off
    for A in range(bs.nshells):
        for B in range(bs.nshells):
            for Cc in range(bs.nshells):
                for D in range(bs.nshells):
                    G[o[A]:o[A + 1], o[B]:o[B + 1], o[Cc]:o[Cc + 1], o[D]:o[D + 1]] = eri_block(bs, A, B, Cc, D)
    return G


def schwarz(bs: Basis) -> np.ndarray:
    Q = np.zeros((bs.nshells, bs.nshells), dtype=np.float64)
    rc = lib(bs.lmax).orc_schwarz(*bs.args(), _p(Q, C.c_double))
    if rc:
        raise ValueError(f"orc_schwarz rc={rc}")
    return Q


def dmax(D) -> float:
    D = np.ascontiguousarray(D, np.float64)
    return float(lib().orc_dmax(_p(D, C.c_double), C.c_int(D.shape[0])))


def dshell(bs: Basis, D) -> np.ndarray:
    """|D|_XY = max over the shell block (X, Y) of max(|D_mu,nu|, |D_nu,mu|): the table of the block-density screen (R-23)."""
    D = np.ascontiguousarray(D, np.float64)
    out = np.zeros((bs.nshells, bs.nshells))
    rc = lib(bs.lmax).orc_dshell(*bs.args(), _p(D, C.c_double), _p(out, C.c_double))
    if rc:
        raise ValueError(f"orc_dshell rc={rc}")
    return out


def jk(bs: Basis, D, tau: float, Q=None, block_density=False):
    """Screened symmetric J/K.  Returns J, K, counts(dict).  block_density: the screen of DESIGN.md R-23
    ((Q_AB*Q_CD)*Dblk(AB|CD) >= tau) instead of the global-Dmax rule."""
    D = np.ascontiguousarray(D, np.float64)
    N = bs.nbf
    assert D.shape == (N, N)
    J = np.zeros((N, N)); K = np.zeros((N, N))
    counts = np.zeros(3, dtype=np.int64); cc = np.zeros(NQCLASS, dtype=np.int64)
    qp = _p(np.ascontiguousarray(Q, np.float64), C.c_double) if Q is not None else None
    fn = lib(bs.lmax).orc_jk_bd if block_density else lib(bs.lmax).orc_jk
    rc = fn(*bs.args(), _p(D, C.c_double), C.c_double(tau), qp, _p(J, C.c_double), _p(K, C.c_double),
            _p(counts, C.c_int64), _p(cc, C.c_int64))
    if rc:
        raise ValueError(f"orc_jk rc={rc}")
    return J, K, {"unique": int(counts[0]), "kept": int(counts[1]), "prim": int(counts[2]), "per_class": cc}


def jk_range(bs: Basis, D, tau: float, Q, pab_lo: int, pab_hi: int):
    """orc_jk's loop over the bra pairs pab = A(A+1)/2+B in [pab_lo, pab_hi) only: long double partial J, K and the
    counts of that range (the partial results of disjoint ranges covering all pairs add up to jk()'s result)."""
    D = np.ascontiguousarray(D, np.float64)
    N = bs.nbf
    J = np.zeros((N, N), dtype=np.longdouble); K = np.zeros((N, N), dtype=np.longdouble)
    counts = np.zeros(3, dtype=np.int64); cc = np.zeros(NQCLASS, dtype=np.int64)
    rc = lib(bs.lmax).orc_jk_range(*bs.args(), _p(D, C.c_double), C.c_double(tau), _p(np.ascontiguousarray(Q, np.float64), C.c_double),
                            C.c_int64(pab_lo), C.c_int64(pab_hi), _p(J, C.c_longdouble), _p(K, C.c_longdouble),
                            _p(counts, C.c_int64), _p(cc, C.c_int64))
    if rc:
        raise ValueError(f"orc_jk_range rc={rc}")
    return J, K, {"unique": int(counts[0]), "kept": int(counts[1]), "prim": int(counts[2]), "per_class": cc}


def count(bs: Basis, Q, Dmax: float, tau: float):
    counts = np.zeros(3, dtype=np.int64); cc = np.zeros(NQCLASS, dtype=np.int64)
    Q = np.ascontiguousarray(Q, np.float64)
    lib(bs.lmax).orc_count(C.c_int(bs.nshells), _p(bs.l, C.c_int32), _p(bs.nprim, C.c_int32), _p(Q, C.c_double),
                    C.c_double(Dmax), C.c_double(tau), _p(counts, C.c_int64), _p(cc, C.c_int64))
    return {"unique": int(counts[0]), "kept": int(counts[1]), "prim": int(counts[2]), "per_class": cc}


def count_bd(bs: Basis, Q, Dsh, tau: float):
    """Kept-quartet counts under the block-density screen (R-23); Dsh = dshell(bs, D)."""
    counts = np.zeros(3, dtype=np.int64); cc = np.zeros(NQCLASS, dtype=np.int64)
    Q = np.ascontiguousarray(Q, np.float64); Dsh = np.ascontiguousarray(Dsh, np.float64)
    lib(bs.lmax).orc_count_bd(C.c_int(bs.nshells), _p(bs.l, C.c_int32), _p(bs.nprim, C.c_int32), _p(Q, C.c_double),
                       _p(Dsh, C.c_double), C.c_double(tau), _p(counts, C.c_int64), _p(cc, C.c_int64))
    return {"unique": int(counts[0]), "kept": int(counts[1]), "prim": int(counts[2]), "per_class": cc}


def jk_brute(bs: Basis, D):
    D = np.ascontiguousarray(D, np.float64)
    N = bs.nbf
    J = np.zeros((N, N)); K = np.zeros((N, N))
    rc = lib(bs.lmax).orc_jk_brute(*bs.args(), _p(D, C.c_double), _p(J, C.c_double), _p(K, C.c_double))
    if rc:
        raise ValueError(f"orc_jk_brute rc={rc}")
    return J, K


def jk_block(bs: Basis, D, tau, Q, Dmax, A, B, want_j=True, want_k=True, with_work=False, Dsh=None):
    """One shell block of J and K from the definition with the screen; Dsh (= dshell(bs, D)) selects the block-density
    rule R-23, otherwise the global rule with Dmax."""
    D = np.ascontiguousarray(D, np.float64); Q = np.ascontiguousarray(Q, np.float64)
    Jb = np.zeros((bs.ncart[A], bs.ncart[B])); Kb = np.zeros((bs.ncart[A], bs.ncart[B]))
    work = np.zeros(2, dtype=np.int64)
    if Dsh is not None:
        Dsh = np.ascontiguousarray(Dsh, np.float64)
        rc = lib(bs.lmax).orc_jk_block_bd(*bs.args(), _p(D, C.c_double), C.c_double(tau), _p(Q, C.c_double), _p(Dsh, C.c_double),
                                   C.c_int(A), C.c_int(B), _p(Jb, C.c_double) if want_j else None,
                                   _p(Kb, C.c_double) if want_k else None, _p(work, C.c_int64))
    else:
        rc = lib(bs.lmax).orc_jk_block(*bs.args(), _p(D, C.c_double), C.c_double(tau), _p(Q, C.c_double), C.c_double(Dmax),
                                C.c_int(A), C.c_int(B), _p(Jb, C.c_double) if want_j else None,
                                _p(Kb, C.c_double) if want_k else None, _p(work, C.c_int64))
    if rc:
        raise ValueError(f"orc_jk_block rc={rc}")
    if with_work:
        return Jb, Kb, (int(work[0]), int(work[1]))
    return Jb, Kb


def energies(D, J, K):
    """E_J = 1/2 tr(DJ), E_K = -1/4 tr(DK) (north_star), accumulated in long double."""
    D = np.asarray(D, np.longdouble)
    return float(0.5 * np.sum(D * np.asarray(J, np.longdouble))), float(-0.25 * np.sum(D * np.asarray(K, np.longdouble)))


def num_threads() -> int:
    return int(lib().orc_num_threads())
