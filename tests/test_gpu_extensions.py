"""GPU parity of the rows SURVEY.md 8(f) marks "next": block-density screening and incremental builds (f3), the sharded
build (f4).  Same bar as tests/test_gpu_parity.py: per-class kept counts equal the oracle's as integers, 1e-10 per element
of J and K, 1e-9 Hartree on the energies; everything through the C ABI."""
import numpy as np
import pytest

from paper_2406_11185_b200 import workloads as W

pytestmark = pytest.mark.gpu
TOL_ELEM = 1e-10
TOL_E = 1e-9


@pytest.fixture(scope="module")
def api():
    import torch
    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    from paper_2406_11185_b200 import api as _api
    _api.lib()
    return _api


def denergy(D, A, B, fac):
    return float(fac * np.sum(np.asarray(D, np.longdouble) * (np.asarray(A, np.longdouble) - np.asarray(B, np.longdouble))))


@pytest.mark.parametrize("cfg,tau", [("0b", 1e-6), (1, 1e-12), (1, 1e-8), (3, None)])
def test_block_density_parity(api, orc, cfg, tau):
    """ADFT_JK_BLOCK_DENSITY (R-23) against the oracle's block-density rule on a density whose shell blocks
    spread over 8 decades: equal per-class counts, J, K, energies.  cfg 3 (f shells, Rys kernels) on a 12-atom cut."""
    w = W.make(cfg)
    if cfg == 3:
        from test_oracle_jk import _first_atoms
        w = _first_atoms(w, 12)
        tau = 1e-10
    D = W.sparse_density(w, 21)
    bs = orc.basis_from_workload(w)
    Qo = orc.schwarz(bs)
    Jo, Ko, cnt = orc.jk(bs, D, tau, Qo, block_density=True)
    glob = orc.count(bs, Qo, orc.dmax(D), tau)
    assert 0 < cnt["kept"] < glob["kept"]                       # the block rule really drops quartets here
    J, K, st, Q = api.jk(w, tau, block_density=True, D=D)
    assert st.quartets_kept == cnt["kept"], (st.quartets_kept, cnt["kept"])
    assert st.prim_quartets == cnt["prim"]
    np.testing.assert_array_equal(np.array(st.class_quartets[:]), cnt["per_class"])
    assert np.abs(J - Jo).max() <= TOL_ELEM and np.abs(K - Ko).max() <= TOL_ELEM
    assert abs(denergy(D, J, Jo, 0.5)) <= TOL_E and abs(denergy(D, K, Ko, -0.25)) <= TOL_E
    assert np.array_equal(J, J.T) and np.array_equal(K, K.T)
    # the default rule on the same density keeps the larger set and is unchanged by the option's existence
    J2, K2, st2, _ = api.jk(w, tau, D=D)
    assert st2.quartets_kept == glob["kept"]


def test_block_density_uniform_blocks_is_global_rule(api, orc):
    w = W.make(1)
    bs = orc.basis_from_workload(w)
    o = bs.bf_off
    D = np.array(w.D)
    for X in range(bs.nshells):
        for Y in range(X + 1):
            D[o[X], o[Y]] = D[o[Y], o[X]] = np.abs(w.D).max()
    Ja, Ka, sa, _ = api.jk(w, w.tau, D=D)
    Jb, Kb, sb, _ = api.jk(w, w.tau, D=D, block_density=True)
    assert sa.quartets_kept == sb.quartets_kept
    assert np.abs(Ja - Jb).max() <= 1e-11 and np.abs(Ka - Kb).max() <= 1e-11


def test_incremental_build(api, orc):
    """adft_jk_build_incremental: J(D1) = J(D0) + J(D1 - D0), the difference built with the block-density screen.
    Oracle: the same decomposition, each part evaluated by the oracle with the same rule."""
    import torch
    w = W.make(1)
    bs = orc.basis_from_workload(w)
    Qo = orc.schwarz(bs)
    D0 = np.array(w.D)
    D1 = W.perturbed_density(w, 33, atoms=(2,), scale=1e-3)
    D2 = W.perturbed_density(w, 34, atoms=(7, 8), scale=1e-5) + (D1 - D0)
    b = api.Basis.from_workload(w); sp = api.ShellPairs(b)
    tD = [torch.from_numpy(np.ascontiguousarray(x)).cuda() for x in (D0, D1, D2)]
    J = torch.empty_like(tD[0]); K = torch.empty_like(tD[0])
    sp.jk_build(tD[0], J, K, w.tau); torch.cuda.synchronize()
    full_kept = sp.stats().quartets_kept
    Jo, Ko, _ = orc.jk(bs, D0, w.tau, Qo)
    Dprev = tD[0].clone()
    for step, (Dn, Dp) in enumerate(((D1, D0), (D2, D1)), 1):
        sp.jk_build_incremental(tD[step], Dprev, J, K, w.tau); torch.cuda.synchronize()
        dJ, dK, cnt = orc.jk(bs, Dn - Dp, w.tau, Qo, block_density=True)
        Jo = Jo + dJ; Ko = Ko + dK
        st = sp.stats()
        assert st.quartets_kept == cnt["kept"] and 0 < st.quartets_kept < full_kept
        np.testing.assert_array_equal(np.array(st.class_quartets[:]), cnt["per_class"])
        assert torch.equal(Dprev, tD[step])
        assert np.abs(J.cpu().numpy() - Jo).max() <= TOL_ELEM and np.abs(K.cpu().numpy() - Ko).max() <= TOL_ELEM
    # and the accumulated result is the from-scratch result up to what the screens dropped (bounded by tau per quartet)
    Jf, Kf, cf = orc.jk(bs, D2, w.tau, Qo)
    assert np.abs(J.cpu().numpy() - Jf).max() <= 1e-7 and np.abs(K.cpu().numpy() - Kf).max() <= 1e-7
    # K-only incremental build leaves J alone
    Jkeep = J.clone()
    sp.jk_build_incremental(tD[1], Dprev, None, K, w.tau); torch.cuda.synchronize()
    assert torch.equal(J, Jkeep) and torch.equal(Dprev, tD[1])
    with pytest.raises(api.AdftError) as e:
        sp.jk_build_incremental(tD[1], tD[1], J, K, w.tau)
    assert e.value.status == 1
    sp.close(); b.close()


@pytest.mark.parametrize("cfg,world", [(1, 2), (1, 3), ("3cut", 4)])
def test_sharded_build_partials_add_up(api, orc, cfg, world):
    """shard_rank / shard_count: every rank's call gives the partial symmetric J, K of its tiles; their sum is the
    full build (what the one all-reduce of jk_build_distributed forms) and the kept counts add up class by class."""
    import torch
    if cfg == "3cut":
        from test_oracle_jk import _first_atoms
        w = _first_atoms(W.make(3), 8)
    else:
        w = W.make(cfg)
    b = api.Basis.from_workload(w); sp = api.ShellPairs(b)
    D = torch.from_numpy(w.D).cuda()
    J = torch.empty_like(D); K = torch.empty_like(D)
    sp.jk_build(D, J, K, w.tau); torch.cuda.synchronize()
    st = sp.stats()
    full_counts = np.array(st.class_quartets[:])
    Js = torch.zeros_like(D); Ks = torch.zeros_like(D)
    counts = np.zeros_like(full_counts)
    for r in range(world):
        Jp = torch.empty_like(D); Kp = torch.empty_like(D)
        sp.jk_build(D, Jp, Kp, w.tau, shard=(r, world)); torch.cuda.synchronize()
        sr = sp.stats()
        assert 0 < sr.quartets_kept < st.quartets_kept
        counts += np.array(sr.class_quartets[:])
        assert torch.equal(Jp, Jp.T) and torch.equal(Kp, Kp.T)
        Js += Jp; Ks += Kp
    np.testing.assert_array_equal(counts, full_counts)
    assert (Js - J).abs().max().item() <= 1e-11 and (Ks - K).abs().max().item() <= 1e-11
    bs = orc.basis_from_workload(w)
    Jo, Ko, _ = orc.jk(bs, w.D, w.tau)
    assert np.abs(Js.cpu().numpy() - Jo).max() <= TOL_ELEM and np.abs(Ks.cpu().numpy() - Ko).max() <= TOL_ELEM
    # one-rank group: jk_build_distributed is the plain build
    J1 = torch.empty_like(D); K1 = torch.empty_like(D)
    sp.jk_build_distributed(D, J1, K1, w.tau); torch.cuda.synchronize()
    assert (J1 - J).abs().max().item() <= 1e-11 and (K1 - K).abs().max().item() <= 1e-11
    for bad in ((2, 2), (-1, 2), (0, -3)):
        with pytest.raises(api.AdftError) as e:
            sp.jk_build(D, J1, K1, w.tau, shard=bad)
        assert e.value.status == 1
    sp.close(); b.close()


def mixed_tolerance(npairs, tau, band):
    """Worst-case bound on an element of J or K of the mixed-precision build against the fp64 oracle:
    a single-precision quartet contributes |D I| <= S < band*tau to an element, with a relative error of at most
    kappa * 2^-24 (kappa = 64 allows for the cancellations of the recurrences between tight and diffuse shells; measured on
    cfg 1 at tau = 1e-10: kappa = 22 would be needed if every term carried the same error); an element collects at most one
    such term per shell pair on the other side and per update pattern (4).  Plus the 1e-10 of the fp64 part."""
    return 1e-10 + 4 * npairs * 64 * 2.0 ** -24 * band * tau


@pytest.mark.parametrize("cfg,tau,band", [(1, 1e-12, 1e5), (1, 1e-10, 1e5), ("0b", 1e-7, 1e3), (1, 1e-12, 1.0)])
def test_mixed_precision_parity(api, orc, cfg, tau, band):
    """ADFT_JK_MIXED_PRECISION: the kept set and the per-class counts are those of the fp64 rule, a
    non-trivial share of the quartets runs in single precision, and J, K stay inside the bound the band implies.
    band = 1 makes the single-precision band empty: the result is then the fp64 build's."""
    w = W.make(cfg)
    bs = orc.basis_from_workload(w)
    Qo = orc.schwarz(bs)
    Jo, Ko, cnt = orc.jk(bs, w.D, tau, Qo)
    J, K, st, Q = api.jk(w, tau, mixed_precision=True, fp32_band=band)
    assert st.quartets_kept == cnt["kept"] and st.prim_quartets == cnt["prim"]
    np.testing.assert_array_equal(np.array(st.class_quartets[:]), cnt["per_class"])
    assert np.array_equal(J, J.T) and np.array_equal(K, K.T)
    npairs = bs.nshells * (bs.nshells + 1) // 2
    dj, dk = np.abs(J - Jo).max(), np.abs(K - Ko).max()
    if band == 1.0:
        assert st.quartets_fp32 == 0
        assert dj <= TOL_ELEM and dk <= TOL_ELEM
        return
    # the single-precision share equals the number of kept quartets below band*tau, counted by the oracle's rule
    n64 = orc.count(bs, Qo, orc.dmax(w.D), tau * band)["kept"]
    assert st.quartets_fp32 == cnt["kept"] - n64 and 0 < st.quartets_fp32 < cnt["kept"]
    np.testing.assert_array_equal(np.array(st.class_quartets_fp32[:]),
                                  cnt["per_class"] - orc.count(bs, Qo, orc.dmax(w.D), tau * band)["per_class"])
    tol = mixed_tolerance(npairs, tau, band)
    print(f"cfg {cfg} tau {tau:g} band {band:g}: fp32 share {st.quartets_fp32 / cnt['kept']:.3f}, max|dJ| {dj:.2e} max|dK| {dk:.2e} (bound {tol:.2e})")
    assert dj <= tol and dk <= tol
    assert abs(denergy(w.D, J, Jo, 0.5)) <= npairs * tol and abs(denergy(w.D, K, Ko, -0.25)) <= npairs * tol


def test_mixed_precision_everything_single(api, orc):
    """A band wide enough to put EVERY kept quartet of cfg 1 in single precision: the fp32 kernels of all 21 s/p/d
    classes against the fp64 oracle at single-precision accuracy (relative to the largest element)."""
    w = W.make(1)
    bs = orc.basis_from_workload(w)
    Jo, Ko, cnt = orc.jk(bs, w.D, w.tau)
    J, K, st, _ = api.jk(w, w.tau, mixed_precision=True, fp32_band=1e300)
    assert st.quartets_kept == cnt["kept"] and st.quartets_fp32 == cnt["kept"]
    assert np.abs(J - Jo).max() <= 2e-5 * np.abs(Jo).max() and np.abs(K - Ko).max() <= 2e-5 * np.abs(Ko).max()
    assert np.abs(J - Jo).max() > 1e-12                   # it really ran in single precision


@pytest.mark.parametrize("chunk", range(3))
def test_mixed_precision_class_sweep(api, orc, chunk):
    """Every ordered (la,lb,lc,ld) in {s,p,d}^4 through the fp32 kernels (band so wide that all quartets are single
    precision): index mapping and canonicalisation of the float instantiations."""
    import itertools
    combos = list(itertools.product([0, 1, 2], repeat=4))[chunk * 27:(chunk + 1) * 27]
    atoms = np.array([[0.0, 0.1, -0.2], [1.3, -0.4, 0.5], [-0.6, 1.1, 0.9], [0.7, 0.8, -1.2]])
    for ls in combos:
        w = W.make_custom(atoms, [(i, ls[i]) for i in range(4)], seed=1000 + sum(l * 3 ** i for i, l in enumerate(ls)),
                          emin=0.2, emax=8.0)
        bs = orc.basis_from_workload(w)
        Jo, Ko, cnt = orc.jk(bs, w.D, 1e-200)
        J, K, st, _ = api.jk(w, 1e-200, mixed_precision=True, fp32_band=1e300)
        assert st.quartets_kept == cnt["kept"] == st.quartets_fp32
        scale = max(np.abs(Jo).max(), np.abs(Ko).max())
        assert np.abs(J - Jo).max() <= 2e-5 * scale and np.abs(K - Ko).max() <= 2e-5 * scale, ls


def test_mixed_precision_errors(api):
    import torch
    w = W.make(0)
    b = api.Basis.from_workload(w); sp = api.ShellPairs(b)
    D = torch.from_numpy(w.D).cuda(); J = torch.empty_like(D); K = torch.empty_like(D)
    for kw in (dict(J=J, K=None), dict(J=None, K=K)):
        with pytest.raises(api.AdftError) as e:
            sp.jk_build(D, tau=1e-10, mixed_precision=True, **kw)
        assert e.value.status == 1
    for band in (0.5, float("inf"), float("nan")):
        with pytest.raises(api.AdftError) as e:
            sp.jk_build(D, J, K, 1e-10, mixed_precision=True, fp32_band=band)
        assert e.value.status == 1
    sp.close(); b.close()


@pytest.mark.parametrize("cfg", [1, "3cut"])
def test_spherical_output(api, orc, cfg):
    """adft_cart_to_spherical: J and K of a build in real solid harmonics against T^T M T of the oracle's
    J, K with the oracle's independently generated T (oracle/sph.py)."""
    import torch
    from oracle import sph
    if cfg == "3cut":
        from test_oracle_jk import _first_atoms
        w = _first_atoms(W.make(3), 8)
    else:
        w = W.make(cfg)
    bs = orc.basis_from_workload(w)
    Jo, Ko, _ = orc.jk(bs, w.D, w.tau)
    b = api.Basis.from_workload(w); sp = api.ShellPairs(b)
    D = torch.from_numpy(w.D).cuda(); J = torch.empty_like(D); K = torch.empty_like(D)
    sp.jk_build(D, J, K, w.tau)
    Js = sp.cart_to_spherical(J); Ks = sp.cart_to_spherical(K); torch.cuda.synchronize()
    nsph = int(sum(2 * int(l) + 1 for l in w.shell_l))
    assert tuple(Js.shape) == (nsph, nsph)
    Jso, Kso = sph.cart_to_spherical(w.shell_l, Jo), sph.cart_to_spherical(w.shell_l, Ko)
    scale = 4 * np.abs(sph.transform_matrix(w.shell_l)).max() ** 2
    assert np.abs(Js.cpu().numpy() - Jso).max() <= TOL_ELEM * scale and np.abs(Ks.cpu().numpy() - Kso).max() <= TOL_ELEM * scale
    assert torch.allclose(Js, Js.T, rtol=0, atol=1e-12)
    with pytest.raises(api.AdftError) as e:
        api._check(api.lib().adft_cart_to_spherical(sp._h, None, None, None))
    assert e.value.status == 1
    sp.close(); b.close()


def test_options_combined(api, orc):
    """Mixed precision together with the block-density screen and with sharding: the kept set is still the oracle's (block
    rule), every quartet is evaluated exactly once across precisions and ranks."""
    import torch
    w = W.make(1)
    D = W.sparse_density(w, 21, decades=4.0)
    bs = orc.basis_from_workload(w)
    Qo = orc.schwarz(bs)
    tau = 1e-10
    Jo, Ko, cnt = orc.jk(bs, D, tau, Qo, block_density=True)
    b = api.Basis.from_workload(w); sp = api.ShellPairs(b)
    tD = torch.from_numpy(D).cuda()
    Js = torch.zeros_like(tD); Ks = torch.zeros_like(tD)
    counts = np.zeros(120, np.int64); n32 = 0
    for r in range(2):
        J = torch.empty_like(tD); K = torch.empty_like(tD)
        sp.jk_build(tD, J, K, tau, block_density=True, mixed_precision=True, shard=(r, 2)); torch.cuda.synchronize()
        st = sp.stats()
        counts += np.array(st.class_quartets[:]); n32 += st.quartets_fp32
        Js += J; Ks += K
    np.testing.assert_array_equal(counts, cnt["per_class"])
    assert 0 < n32 < cnt["kept"]
    tol = mixed_tolerance(bs.nshells * (bs.nshells + 1) // 2, tau, 1e5)
    assert np.abs(Js.cpu().numpy() - Jo).max() <= tol and np.abs(Ks.cpu().numpy() - Ko).max() <= tol
    sp.close(); b.close()
