"""Pins for the oracle's block-density screen (reading R-23).  CPU only.

The rule: keep a unique quartet iff (Q_AB*Q_CD) * Dblk >= tau with
Dblk = max(|D|_AB, |D|_CD, |D|_AC, |D|_AD, |D|_BC, |D|_BD), |D|_XY the largest |D| element of the shell block.
Pinned here against things that do not go through the oracle's own loop: the masked contraction of the full
integral tensor written with numpy (P17b), the special case of a density whose shell blocks all have the same maximum,
where the rule IS the global one (P17a), and the set relations the definition implies (P17c).
"""
import numpy as np
import pytest

from paper_2406_11185_b200 import workloads as W


def _dshell_numpy(bs, D):
    o = bs.bf_off
    out = np.zeros((bs.nshells, bs.nshells))
    for X in range(bs.nshells):
        for Y in range(bs.nshells):
            out[X, Y] = max(np.abs(D[o[X]:o[X + 1], o[Y]:o[Y + 1]]).max(), np.abs(D[o[Y]:o[Y + 1], o[X]:o[X + 1]]).max())
    return out


_sparse_density = W.sparse_density


@pytest.mark.parametrize("cfg", [0, "0b", 1])
def test_p17d_dshell_is_the_block_maximum(orc, cfg):
    w = W.make(cfg)
    bs = orc.basis_from_workload(w)
    D = _sparse_density(w, 5)
    D[0, -1] *= 3.0                       # an unsymmetric D: the table takes both triangles
    np.testing.assert_array_equal(orc.dshell(bs, D), _dshell_numpy(bs, D))


@pytest.mark.parametrize("cfg", [0, "0b"])
def test_p17b_block_rule_equals_masked_tensor_contraction(orc, cfg):
    """J and K under the block rule against Eq. 1 contracted with numpy over the full integral tensor, every ORDERED
    shell quartet masked by the rule written out here (no symmetry, no canonical order, no oracle loop)."""
    w = W.make(cfg)
    bs = orc.basis_from_workload(w)
    D = _sparse_density(w, 7)
    Q = orc.schwarz(bs)
    G = orc.eri_tensor(bs)
    Dsh = _dshell_numpy(bs, D)
    ns, o, N = bs.nshells, bs.bf_off, bs.nbf
    prod = np.sort((Q[:, :, None, None] * Q[None, None, :, :]).ravel())
    for tau in (0.0, float(prod[len(prod) // 3] * np.median(Dsh)), float(prod[2 * len(prod) // 3] * np.median(Dsh))):
        mask = np.zeros((N, N, N, N))
        kept_ordered = 0
        for A in range(ns):
            for B in range(ns):
                for Cc in range(ns):
                    for Dd in range(ns):
                        dblk = max(Dsh[A, B], Dsh[Cc, Dd], Dsh[A, Cc], Dsh[A, Dd], Dsh[B, Cc], Dsh[B, Dd])
                        if (Q[A, B] * Q[Cc, Dd]) * dblk >= tau:
                            mask[o[A]:o[A + 1], o[B]:o[B + 1], o[Cc]:o[Cc + 1], o[Dd]:o[Dd + 1]] = 1.0
                            kept_ordered += 1
        Jref = np.einsum("ls,mnls->mn", D, G * mask)
        Kref = np.einsum("ns,mnls->ml", D, G * mask)
        J, K, cnt = orc.jk(bs, D, tau, Q, block_density=True)
        scale = max(np.abs(Jref).max(), np.abs(Kref).max(), 1e-300)
        assert np.abs(J - Jref).max() <= 1e-13 * scale and np.abs(K - Kref).max() <= 1e-13 * scale
        if tau > 0.0:
            assert 0 < cnt["kept"] < cnt["unique"] and 0 < kept_ordered < ns ** 4       # the mask really cuts
        c2 = orc.count_bd(bs, Q, orc.dshell(bs, D), tau)
        assert c2["kept"] == cnt["kept"] and c2["prim"] == cnt["prim"]
        np.testing.assert_array_equal(c2["per_class"], cnt["per_class"])
        # the per-block definition (used where the full oracle is too slow) gives the same blocks
        for (A, B) in ((0, 0), (ns - 1, 1), (2, ns - 2)):
            Jb, Kb = orc.jk_block(bs, D, tau, Q, 0.0, A, B, Dsh=orc.dshell(bs, D))
            assert np.abs(Jb - J[o[A]:o[A + 1], o[B]:o[B + 1]]).max() <= 1e-13 * scale
            assert np.abs(Kb - K[o[A]:o[A + 1], o[B]:o[B + 1]]).max() <= 1e-13 * scale


def test_p17a_uniform_block_maxima_reduce_to_the_global_rule(orc):
    """If every shell block of D has the same largest element, Dblk = Dmax for every quartet and the rule is R-6/R-7."""
    w = W.make(1)
    bs = orc.basis_from_workload(w)
    o = bs.bf_off
    D = np.array(w.D)
    dm = np.abs(D).max()
    for X in range(bs.nshells):
        for Y in range(X + 1):
            D[o[X], o[Y]] = D[o[Y], o[X]] = dm          # one element of every block at the global maximum
    Q = orc.schwarz(bs)
    J0, K0, c0 = orc.jk(bs, D, w.tau, Q)
    J1, K1, c1 = orc.jk(bs, D, w.tau, Q, block_density=True)
    assert c0["kept"] == c1["kept"] and 0 < c0["kept"] < c0["unique"]
    np.testing.assert_array_equal(c0["per_class"], c1["per_class"])
    assert np.abs(J0 - J1).max() <= 1e-13 * np.abs(J0).max() and np.abs(K0 - K1).max() <= 1e-13 * np.abs(K0).max()


def test_p17c_block_rule_keeps_a_subset_and_is_monotone(orc):
    w = W.make(1)
    bs = orc.basis_from_workload(w)
    D = _sparse_density(w, 11)
    Q = orc.schwarz(bs)
    Dsh = orc.dshell(bs, D)
    assert Dsh.max() == orc.dmax(D)
    last = None
    for tau in (0.0, 1e-14, 1e-12, 1e-10, 1e-8, 1e-6):
        g = orc.count(bs, Q, orc.dmax(D), tau)
        b = orc.count_bd(bs, Q, Dsh, tau)
        assert b["unique"] == g["unique"] and b["kept"] <= g["kept"]
        assert (b["per_class"] <= g["per_class"]).all()
        if tau == 0.0:
            assert b["kept"] == b["unique"]
        if last is not None:
            assert b["kept"] <= last
        last = b["kept"]
    assert orc.count_bd(bs, Q, Dsh, 1e-10)["kept"] < orc.count(bs, Q, orc.dmax(D), 1e-10)["kept"]
    # dropping what the block rule drops changes J, K by no more than the bound it enforces
    tau = 1e-10
    Jg, Kg, cg = orc.jk(bs, D, tau, Q)
    Jb, Kb, cb = orc.jk(bs, D, tau, Q, block_density=True)
    dropped = cg["kept"] - cb["kept"]
    assert dropped > 0
    assert np.abs(Jg - Jb).max() <= 4 * dropped * tau and np.abs(Kg - Kb).max() <= 4 * dropped * tau
