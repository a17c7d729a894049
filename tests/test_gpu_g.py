"""GPU parity of the g-shell classes (SURVEY.md 8(f2); PAPER.md:191 "110 tests have up to g functions", :222): the 65
quartet classes with a g shell run through the block-cooperative Rys kernels with up to 9 roots.  Same bar as
tests/test_gpu_parity.py: Schwarz table to 1e-12 relative, per-class kept counts equal to the oracle's as integers,
1e-10 per element of J and K, 1e-9 Hartree on the energies.  The oracle for l = 4 is oracle/liboracle_g.so (pins in
tests/test_oracle_g.py)."""
import itertools

import numpy as np
import pytest

from paper_2406_11185_b200 import workloads as W
from test_gpu_parity import check_full, WIDE_ATOMS

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def api():
    import torch
    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    from paper_2406_11185_b200 import api as _api
    _api.lib()
    return _api


G_COMBOS = [c for c in itertools.product([0, 1, 2, 3, 4], repeat=4) if 4 in c]          # 369 ordered combinations
ATOMS = np.array([[0.0, 0.1, -0.2], [1.3, -0.4, 0.5], [-0.6, 1.1, 0.9], [0.7, 0.8, -1.2]])


@pytest.mark.parametrize("chunk", range(9))
def test_class_sweep_g_orderings(api, orc, chunk):
    """4 atoms, one shell each, every ordered (la,lb,lc,ld) in {s,p,d,f,g}^4 that contains a g shell: all 65 g classes in
    every orientation (pair swaps, bra/ket swap), random contraction depth 1..3."""
    for ls in G_COMBOS[chunk * 41:(chunk + 1) * 41]:
        rng = np.random.default_rng(sum(l * 5 ** i for i, l in enumerate(ls)))
        w = W.make_custom(ATOMS, [(i, ls[i]) for i in range(4)], seed=11000 + sum(l * 5 ** i for i, l in enumerate(ls)),
                          emin=0.2, emax=8.0, nprim=int(rng.integers(1, 4)))
        check_full(api, orc, w, tau=0.0)


@pytest.mark.parametrize("ls", [(4, 4, 4, 4), (4, 0, 2, 4), (3, 4, 4, 1), (4, 4, 0, 0), (0, 4, 3, 3), (4, 2, 4, 2), (1, 4, 2, 3),
                                (4, 3, 4, 4)])
def test_g_wide_exponents(api, orc, ls):
    """Exponents log-uniform in [0.05, 5000], atoms 3.7-11.3 bohr apart: tight g shells next to distant diffuse ones."""
    w = W.make_custom(WIDE_ATOMS, [(i, ls[i]) for i in range(4)], seed=13000 + sum(l * 5 ** i for i, l in enumerate(ls)),
                      emin=0.05, emax=5000.0, nprim=2)
    check_full(api, orc, w, tau=0.0)


@pytest.mark.parametrize("ls", [(4, 4), (4, 0), (4, 2), (1, 4), (3, 4)])
def test_g_coincident_shells(api, orc, ls):
    """Two shells on one atom and a copy on a second: A = B, C = D, AB = CD weights and AB = 0 geometry at g level."""
    atoms = np.array([[0.0, 0.0, 0.0], [0.9, -0.7, 1.1]])
    spec = [(0, ls[0]), (0, ls[1]), (1, ls[0]), (1, ls[1])]
    w = W.make_custom(atoms, spec, seed=1500 + 10 * ls[0] + ls[1], emin=0.2, emax=8.0, nprim=2)
    check_full(api, orc, w, tau=0.0)
    check_full(api, orc, w, tau=1e-6)


def test_g_mixed_basis_screened(api, orc):
    """Seven atoms with s, p, d, f and g shells (24 shells, 162 functions), tau = 1e-10: the screen, the class histogram
    over the 120 classes and the digestion of blocks of mixed shape in one build."""
    rng = np.random.default_rng(2406)
    atoms = rng.uniform(-4.5, 4.5, size=(7, 3))
    spec = []
    for a in range(7):
        spec += [(a, 0), (a, 1), (a, int(rng.integers(2, 5)))]
    spec += [(0, 4), (3, 4), (6, 3)]
    w = W.make_custom(atoms, spec, seed=2407, emin=0.08, emax=400.0, tau=1e-10)
    J, K, st = check_full(api, orc, w)
    assert 0 < st.quartets_kept < st.quartets_unique
    assert sum(1 for c in st.class_quartets[55:] if c) >= 20          # many g classes really ran


def test_g_spherical_output(api, orc):
    """adft_cart_to_spherical on a basis with g shells: the l = 4 harmonics of the library's table against oracle/sph.py."""
    import torch
    from oracle import sph
    w = W.make_custom(ATOMS, [(0, 4), (1, 2), (2, 4), (3, 1)], seed=31, emin=0.2, emax=8.0, nprim=2)
    bs = orc.basis_from_workload(w)
    Jo, Ko, _ = orc.jk(bs, w.D, 0.0)
    b = api.Basis.from_workload(w); sp = api.ShellPairs(b)
    D = torch.from_numpy(w.D).cuda(); J = torch.empty_like(D); K = torch.empty_like(D)
    sp.jk_build(D, J, K, 0.0)
    Js = sp.cart_to_spherical(J).cpu().numpy(); Ks = sp.cart_to_spherical(K).cpu().numpy()
    assert Js.shape == (9 + 5 + 9 + 3, 9 + 5 + 9 + 3)
    T = sph.transform_matrix(w.shell_l)
    tol = 4e-10 * np.abs(T).max() ** 2
    assert np.abs(Js - T.T @ Jo @ T).max() <= tol and np.abs(Ks - T.T @ Ko @ T).max() <= tol
    sp.close(); b.close()


def test_l5_is_rejected(api):
    w = W.make(0)
    sh = w.shells_struct().copy(); sh[0, 1] = 5
    with pytest.raises(api.AdftError) as e:
        api.Basis(w.atoms, sh, w.exponents, w.coefficients)
    assert e.value.status == 2
