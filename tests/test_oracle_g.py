"""Pins of the oracle at L = 4 (g shells).  CPU only.

liboracle_g.so is oracle/jk_oracle.c compiled with -DLMAX_SHELL=4: the recurrences are the same code, only table sizes
grow.  What is pinned here is therefore (a) that the larger tables are wired correctly (component tables to degree 8,
Boys orders to 16, the 15^4 block, 120 classes) and (b) the g-level values themselves, against references that share
nothing with Obara-Saika: the one-centre closed form (P6), the 50-digit McMurchie-Davidson evaluation (P16), the
normaliser's quadrature (P3'), and the invariances of the definition (P8, P9).
"""
import itertools

import mpmath as mp
import numpy as np
import pytest

from test_oracle_p16 import _compare
from test_oracle_pins import comps, p6_ref, prim_basis

mp.mp.dps = 50


def test_g_library_is_a_second_build_of_the_same_source(orc):
    assert orc.lib(3).orc_lmax() == 3 and orc.lib(4).orc_lmax() == 4
    assert orc.lib(3).orc_nqclass() == 55 and orc.lib(4).orc_nqclass() == 120 == orc.NQCLASS


def test_g_build_reproduces_the_f_build(orc):
    """The l <= 3 results do not depend on which build evaluates them (same recurrences, other table strides)."""
    from paper_2406_11185_b200 import workloads as W
    w = W.make("0b")
    bs = orc.basis_from_workload(w)
    J3, K3, c3 = orc.jk(bs, w.D, w.tau)
    bs.lmax = 4                                   # route the same basis through liboracle_g.so
    J4, K4, c4 = orc.jk(bs, w.D, w.tau)
    assert c3["kept"] == c4["kept"] and np.array_equal(c3["per_class"], c4["per_class"])
    assert np.abs(J3 - J4).max() <= 1e-14 * np.abs(J3).max() and np.abs(K3 - K4).max() <= 1e-14 * np.abs(K3).max()
    at = np.array([[0.0, 0.1, -0.2], [1.3, -0.4, 0.5], [-0.6, 1.1, 0.9], [0.7, 0.8, -1.2]])
    wf = W.make_custom(at, [(0, 3), (1, 2), (2, 3), (3, 1)], seed=4, emin=0.2, emax=8.0)
    b3 = orc.basis_from_workload(wf)
    blk3 = orc.eri_block(b3, 0, 1, 2, 3)
    b3.lmax = 4
    np.testing.assert_allclose(orc.eri_block(b3, 0, 1, 2, 3), blk3, rtol=1e-13, atol=1e-16)


def test_g_normaliser_unit_self_overlap(orc):
    rng = np.random.default_rng(44)
    n = 4
    e = np.exp(rng.uniform(np.log(0.1), np.log(100), size=n))
    c = rng.uniform(0.1, 1, size=n)
    d = orc.normalize([4], [n], [0], e, c)
    S = mp.mpf(0)
    for i in range(n):
        for j in range(n):
            p = mp.mpf(e[i]) + mp.mpf(e[j])
            ix = mp.quad(lambda x: x ** 8 * mp.exp(-p * x * x), [-mp.inf, 0, mp.inf])
            iy = mp.quad(lambda x: mp.exp(-p * x * x), [-mp.inf, 0, mp.inf])
            S += d[i] * d[j] * ix * iy * iy
    assert float(S) == pytest.approx(1.0, rel=1e-13)


@pytest.mark.parametrize("side", ["bra", "ket"])
@pytest.mark.parametrize("la,lb", [(4, 0), (4, 2), (4, 4), (3, 4), (1, 4)])
def test_g_p6_one_centre_products(orc, side, la, lb):
    """(a b|ss) on one centre against the closed form (radial quadrature x double-factorial angular factor), product
    degree up to 8: the VRR to degree la+lb, the HRR with A = B, and by bra<->ket symmetry the ket VRR."""
    zeta, eta, za = 1.3, 0.9, 0.4
    specs = [(0, la, za), (0, lb, zeta - za), (0, 0, 0.25), (0, 0, eta - 0.25)]
    bs = prim_basis(orc, [[0.3, -0.2, 0.7]], specs)
    blk = orc.eri_block(bs, 0, 1, 2, 3)[:, :, 0, 0] if side == "bra" else orc.eri_block(bs, 2, 3, 0, 1)[0, 0, :, :]
    for ia, a in enumerate(comps(la)):
        for ib, b in enumerate(comps(lb)):
            ref = p6_ref(a[0] + b[0], a[1] + b[1], a[2] + b[2], mp.mpf(zeta), mp.mpf(eta))
            assert blk[ia, ib] == pytest.approx(ref, rel=2e-12, abs=1e-14), (a, b)


@pytest.mark.parametrize("ls", [(4, 1, 2, 4), (4, 4, 4, 4), (2, 4, 4, 3)])
def test_g_p16_primitive_quartet_tight_diffuse(orc, ls):
    """Four centres, alpha = 4595.251 on A, 0.05 on B (10.9 bohr away), 2019.87 on C, 0.3 on D, against the independent
    50-digit McMurchie-Davidson evaluation of tests/test_oracle_p16.py."""
    res = _compare(orc, ls, [[4595.251], [0.05], [2019.87], [0.3]], [[1.0], [1.0], [1.0], [1.0]], nsample=16, seed=26)
    for ld, (wabs, wrel, scale) in res.items():
        assert scale > 0
        assert wabs <= (1e-15 if ld else 1e-12), (ld, wabs, wrel)
        assert wrel <= (1e-14 if ld else 1e-11), (ld, wabs, wrel)


def test_g_p16_contracted_quartet(orc):
    exps = [[4595.251, 3.1], [38.639, 0.05], [2019.87, 0.246], [1.7, 0.3]]
    cofs = [[0.75, 0.4], [1.0, 0.77], [0.53, 0.22], [0.6, 0.4]]
    res = _compare(orc, (4, 2, 3, 4), exps, cofs, nsample=8, seed=27)
    for ld, (wabs, wrel, scale) in res.items():
        assert wabs <= (1e-15 if ld else 1e-12), (ld, wabs, wrel)
        assert wrel <= (1e-14 if ld else 1e-11), (ld, wabs, wrel)


@pytest.mark.parametrize("ls", [(4, 2, 3, 1), (4, 4, 4, 4), (0, 4, 4, 0)])
def test_g_p9_eightfold_symmetry(orc, ls):
    """(ab|cd) = (ba|cd) = (ab|dc) = (cd|ab) and their combinations on four centres, contracted shells."""
    from paper_2406_11185_b200 import workloads as W
    at = np.array([[0.0, 0.1, -0.2], [1.3, -0.4, 0.5], [-0.6, 1.1, 0.9], [0.7, 0.8, -1.2]])
    w = W.make_custom(at, [(i, ls[i]) for i in range(4)], seed=900 + sum(ls), emin=0.2, emax=30.0, nprim=2)
    bs = orc.basis_from_workload(w)
    ref = orc.eri_block(bs, 0, 1, 2, 3, long_double=True)
    scale = float(np.abs(ref).max())
    perms = {(1, 0, 2, 3): (1, 0, 2, 3), (0, 1, 3, 2): (0, 1, 3, 2), (1, 0, 3, 2): (1, 0, 3, 2), (2, 3, 0, 1): (2, 3, 0, 1),
             (3, 2, 0, 1): (3, 2, 0, 1), (2, 3, 1, 0): (2, 3, 1, 0), (3, 2, 1, 0): (3, 2, 1, 0)}
    for order in perms:
        blk = orc.eri_block(bs, *order, long_double=True)
        back = np.transpose(blk, np.argsort(order))
        assert float(np.abs(back - ref).max()) <= 1e-13 * scale, order


def test_g_jk_counts_and_brute_force(orc):
    """Two atoms with s, p and g shells: the symmetric screened scheme equals Eq. 1 written out (orc_jk_brute), the class
    histogram uses the 120-class indexing, Schwarz bounds are the block diagonal."""
    from paper_2406_11185_b200 import workloads as W
    at = np.array([[0.0, 0.0, 0.0], [1.4, 0.6, -0.9]])
    w = W.make_custom(at, [(0, 4), (0, 1), (1, 0), (1, 4)], seed=77, emin=0.3, emax=6.0, nprim=2)
    bs = orc.basis_from_workload(w)
    assert bs.nbf == 15 + 3 + 1 + 15
    J, K, cnt = orc.jk(bs, w.D, 0.0)
    Jb, Kb = orc.jk_brute(bs, w.D)
    scale = max(np.abs(Jb).max(), np.abs(Kb).max())
    assert np.abs(J - Jb).max() <= 1e-13 * scale and np.abs(K - Kb).max() <= 1e-13 * scale
    assert cnt["kept"] == cnt["unique"] == 55 and cnt["per_class"].sum() == 55
    pc = lambda a, b: max(a, b) * (max(a, b) + 1) // 2 + min(a, b)
    qc = lambda X, Y: max(X, Y) * (max(X, Y) + 1) // 2 + min(X, Y)
    assert cnt["per_class"][qc(pc(4, 4), pc(4, 4))] == 6          # (gg|gg): pairs (0,0), (3,0), (3,3) -> 6 unique quartets
    Q = orc.schwarz(bs)
    blk = orc.eri_block(bs, 0, 3, 0, 3)
    assert Q[0, 3] == pytest.approx(np.sqrt(max(abs(blk[i, j, i, j]) for i in range(15) for j in range(15))), rel=1e-13)
