"""Pins for the oracle's J/K assembly and screening.  CPU only."""
import json
import os

import numpy as np
import pytest

from paper_2406_11185_b200 import workloads as W

GOLD = json.load(open(os.path.join(os.path.dirname(__file__), "golden", "survey_pins.json")))


def test_p5b_jk_energies_q(orc):
    g5, g = GOLD["P5"], GOLD["P5b"]
    e, c = g5["exponents"], g5["coefficients"]
    sl, sn, so = [0, 0], [3, 3], [0, 3]
    cf = orc.normalize(sl, sn, so, e + e, c + c)
    bs = orc.Basis([[0, 0, 0], [0, 0, g5["R"]]], [0, 1], sl, sn, so, e + e, cf)
    D = np.array(g["D"])
    J, K, cnt = orc.jk(bs, D, 0.0)
    assert cnt["unique"] == cnt["kept"] == 6
    assert J[0, 0] == pytest.approx(g["J11"], abs=2e-10) and J[1, 1] == pytest.approx(g["J11"], abs=2e-10)
    assert J[0, 1] == pytest.approx(g["J12"], abs=2e-10) and J[1, 0] == pytest.approx(g["J12"], abs=2e-10)
    assert K[0, 0] == pytest.approx(g["K11"], abs=2e-10) and K[0, 1] == pytest.approx(g["K12"], abs=2e-10)
    EJ, EK = orc.energies(D, J, K)
    assert EJ == pytest.approx(g["EJ"], abs=2e-10) and EK == pytest.approx(g["EK"], abs=2e-10)
    Q = orc.schwarz(bs)
    assert Q[0, 0] == pytest.approx(g["Q11"], abs=2e-10) and Q[1, 0] == pytest.approx(g["Q21"], abs=2e-10)


def _first_atoms(w, natoms):
    keep = [i for i in range(w.nshells) if w.shell_atom[i] < natoms]
    off = w.bf_offsets()
    bfs = np.concatenate([np.arange(off[i], off[i + 1]) for i in keep])
    sub = W.Workload(w.name + f"_first{natoms}", w.atoms[:natoms], w.shell_atom[keep], w.shell_l[keep],
                     w.shell_nprim[keep], w.shell_off[keep], w.exponents, w.coefficients,
                     np.ascontiguousarray(w.D[np.ix_(bfs, bfs)]), w.tau)
    return sub


@pytest.mark.parametrize("cfg", [0, "0b", "1cut"])
def test_p12_symmetric_scheme_equals_definition(orc, cfg):
    w = _first_atoms(W.make(1), 3) if cfg == "1cut" else W.make(cfg)
    bs = orc.basis_from_workload(w)
    J, K, cnt = orc.jk(bs, w.D, 0.0)
    npair = bs.nshells * (bs.nshells + 1) // 2
    assert cnt["unique"] == cnt["kept"] == npair * (npair + 1) // 2          # P14: tau = 0 keeps all
    Jb, Kb = orc.jk_brute(bs, w.D)
    scale = max(np.abs(Jb).max(), np.abs(Kb).max())
    assert np.abs(J - Jb).max() <= 1e-13 * scale
    assert np.abs(K - Kb).max() <= 1e-13 * scale
    # and against plain einsum over the full tensor (the textbook contraction of Eq. 1)
    if bs.nbf <= 30:
        G = orc.eri_tensor(bs)
        np.testing.assert_allclose(J, np.einsum("ls,mnls->mn", w.D, G), atol=1e-13 * scale)
        np.testing.assert_allclose(K, np.einsum("ns,mnls->ml", w.D, G), atol=1e-13 * scale)
    # P9: symmetry of the outputs
    assert np.abs(J - J.T).max() <= 1e-14 * scale and np.abs(K - K.T).max() <= 1e-14 * scale


@pytest.fixture(scope="module")
def cfg1(orc):
    w = W.make(1)
    bs = orc.basis_from_workload(w)
    Q = orc.schwarz(bs)
    J, K, cnt = orc.jk(bs, w.D, w.tau, Q)
    return w, bs, Q, J, K, cnt


def test_cfg1_sizes(cfg1):
    w, bs, Q, J, K, cnt = cfg1
    assert bs.nbf == 100 and bs.nshells == 45
    assert cnt["unique"] == 1035 * 1036 // 2
    assert 0 < cnt["kept"] < cnt["unique"]
    assert cnt["per_class"].sum() == cnt["kept"]


def test_p9_p11_symmetry_and_positivity(orc, cfg1):
    w, bs, Q, J, K, cnt = cfg1
    scale = np.abs(J).max()
    assert np.abs(J - J.T).max() <= 1e-14 * scale and np.abs(K - K.T).max() <= 1e-14 * scale
    EJ, EK = orc.energies(w.D, J, K)
    assert EJ > 0 and EK < 0                      # tr(DJ) >= 0 for any D; tr(DK) >= 0 for PSD D
    rng = np.random.default_rng(11)
    S = rng.standard_normal(w.D.shape); S = S + S.T          # indefinite symmetric D
    J2, _, _ = orc.jk(bs, S, 0.0, Q)
    assert np.sum(S * J2) > 0


def test_p14_screening_bounds(orc, cfg1):
    w, bs, Q, J, K, cnt = cfg1
    J0, K0, c0 = orc.jk(bs, w.D, 0.0, Q)
    dm = orc.dmax(w.D)
    prev = c0["kept"]
    for tau in [1e-14, 1e-12, 1e-9, 1e-6]:
        c = orc.count(bs, Q, dm, tau)
        assert c["kept"] <= prev and c["per_class"].sum() == c["kept"]
        prev = c["kept"]
    assert orc.count(bs, Q, dm, w.tau)["kept"] == cnt["kept"]
    nskip = c0["kept"] - cnt["kept"]
    # every skipped quartet contributes < tau per update, <= 4 updates per element per integral of the quartet
    assert np.abs(J - J0).max() <= w.tau * nskip * 4 and np.abs(K - K0).max() <= w.tau * nskip * 4
    assert np.abs(J - J0).max() > 0 or nskip == 0


def test_block_oracle_equals_full(orc, cfg1):
    """orc_jk_block (definition + screen, used for sampled parity at cfg 2-4) reproduces blocks of orc_jk."""
    w, bs, Q, J, K, cnt = cfg1
    dm = orc.dmax(w.D)
    o = bs.bf_off
    rng = np.random.default_rng(21)
    for _ in range(6):
        A, B = rng.integers(0, bs.nshells, size=2)
        Jb, Kb = orc.jk_block(bs, w.D, w.tau, Q, dm, int(A), int(B))
        np.testing.assert_allclose(Jb, J[o[A]:o[A + 1], o[B]:o[B + 1]], atol=2e-12)
        np.testing.assert_allclose(Kb, K[o[A]:o[A + 1], o[B]:o[B + 1]], atol=2e-12)


def test_workload_shapes():
    assert W.make(0).nbf == 13 and W.make("0b").nbf == 13
    assert W.make(2).nbf == 500 and W.make(3).nbf == 940
    w4 = W.make(4)
    assert w4.nbf == 2500 and w4.nshells == 1200 and abs(np.trace(w4.D) - 600) < 1e-9
    d = np.linalg.norm(w4.atoms[:, None] - w4.atoms[None], axis=-1) + 10 * np.eye(300)
    assert d.min() >= 2.0
    w0 = W.make(0)
    assert np.allclose(w0.exponents[:3], w0.exponents[3:6])      # R-14: one shared set
    for cfg in (1, 2):
        w = W.make(cfg)
        assert np.allclose(w.D, w.D.T) and w.exponents.min() >= 0.05 and w.exponents.max() <= 5e3
    assert np.array_equal(W.make(2).atoms, W.make(3).atoms)      # R-17: cfg 3 shares cfg 2 geometry
