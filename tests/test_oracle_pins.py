"""Pins for the oracle's integral core.  CPU only.

Nothing here compares the oracle with itself through the same route: references are closed forms
evaluated with mpmath / scipy, numerical quadrature, finite differences, or exact symmetries.
"""
import itertools
import json
import os

import mpmath as mp
import numpy as np
import pytest

from paper_2406_11185_b200 import workloads as W

GOLD = json.load(open(os.path.join(os.path.dirname(__file__), "golden", "survey_pins.json")))
mp.mp.dps = 40


def comps(l):
    """Component order inside a shell: lx descending, then ly descending (SURVEY R-3)."""
    return [(x, y, l - x - y) for x in range(l, -1, -1) for y in range(l - x, -1, -1)]


def prim_basis(orc, centers, specs):
    """specs = [(center_index, l, exponent)], unnormalised single primitives with coefficient 1."""
    n = len(specs)
    return orc.Basis(np.array(centers, float), [s[0] for s in specs], [s[1] for s in specs], [1] * n,
                     list(range(n)), [s[2] for s in specs], [1.0] * n)


# ---------------------------------------------------------------- P1 Boys
def boys_ref(m, T):
    if T == 0:
        return mp.mpf(1) / (2 * m + 1)
    return mp.hyp1f1(m + mp.mpf(1) / 2, m + mp.mpf(3) / 2, -mp.mpf(T)) / (2 * m + 1)


def test_p1_boys_golden(orc):
    for m, T, val in GOLD["boys"]:
        assert orc.boys(12, T)[m] == pytest.approx(val, rel=2e-14)


def test_p1_boys_special_functions(orc):
    Ts = [0.0, 1e-9, 1e-3, 0.1, 0.5, 1.0, 3.3, 7.7, 12.0, 20.0, 29.9, 34.9, 34.999999, 35.0, 35.000001, 36.0, 50.0,
          80.0, 120.0, 200.0]
    for T in Ts:
        F = orc.boys(12, T)
        for m in range(13):
            ref = float(boys_ref(m, T))
            assert F[m] == pytest.approx(ref, rel=5e-14), (m, T)
    # F_m(0) = 1/(2m+1); F_0 = 1/2 sqrt(pi/T) erf(sqrt T); large-T asymptote
    for m in range(13):
        assert orc.boys(12, 0.0)[m] == pytest.approx(1.0 / (2 * m + 1), rel=1e-15)
    for T in [0.3, 4.0, 33.0, 90.0]:
        assert orc.boys(0, T)[0] == pytest.approx(float(mp.sqrt(mp.pi / T) * mp.erf(mp.sqrt(T)) / 2), rel=1e-14)
    T = 190.0
    for m in range(13):
        asym = float(mp.fac2(2 * m - 1) / mp.mpf(2) ** (m + 1) * mp.sqrt(mp.pi / mp.mpf(T) ** (2 * m + 1)))
        assert orc.boys(12, T)[m] == pytest.approx(asym, rel=1e-13)


def test_p1_boys_lower_mmax_consistent(orc):
    """F_m must not depend on the mmax the recursion was started from (catches recursion index slips)."""
    for T in [0.2, 9.0, 34.0, 36.0, 77.0]:
        F12 = orc.boys(12, T)
        for mmax in [0, 1, 4, 7]:
            np.testing.assert_allclose(orc.boys(mmax, T), F12[:mmax + 1], rtol=2e-14)


# ---------------------------------------------------------------- P2-P4 s-type closed forms
def ssss_closed(za, zb, zc, zd, A, B, C, D):
    A, B, C, D = [mp.matrix(v) for v in (A, B, C, D)]
    zeta, eta = mp.mpf(za) + zb, mp.mpf(zc) + zd
    P = (za * A + zb * B) / zeta
    Q = (zc * C + zd * D) / eta
    n2 = lambda v: sum(x * x for x in v)
    T = zeta * eta / (zeta + eta) * n2(P - Q)
    F0 = mp.mpf(1) if T == 0 else mp.sqrt(mp.pi / T) * mp.erf(mp.sqrt(T)) / 2
    return (2 * mp.pi ** 2.5 / (zeta * eta * mp.sqrt(zeta + eta)) * mp.exp(-za * zb / zeta * n2(A - B))
            * mp.exp(-zc * zd / eta * n2(C - D)) * F0)


def test_p2_ssss_primitive_closed_form(orc):
    rng = np.random.default_rng(5)
    for _ in range(20):
        cen = rng.normal(0, 1.5, size=(4, 3))
        z = np.exp(rng.uniform(np.log(0.05), np.log(50), size=4))
        bs = prim_basis(orc, cen, [(i, 0, z[i]) for i in range(4)])
        val = orc.eri_block(bs, 0, 1, 2, 3)[0, 0, 0, 0]
        assert val == pytest.approx(float(ssss_closed(*z, *cen)), rel=2e-13)


def test_p3_one_centre(orc):
    a = GOLD["P3"]["alpha"]
    cf = orc.normalize([0], [1], [0], [a], [1.0])
    bs = orc.Basis([[0, 0, 0]], [0], [0], [1], [0], [a], cf)
    v = orc.eri_block(bs, 0, 0, 0, 0)[0, 0, 0, 0]
    assert v == pytest.approx(GOLD["P3"]["value"], rel=1e-13)
    assert v == pytest.approx(2 * np.sqrt(a / np.pi), rel=1e-14)


def test_p4_two_centre(orc):
    g = GOLD["P4"]
    a, b, R = g["a"], g["b"], g["R"]
    cf = orc.normalize([0, 0], [1, 1], [0, 1], [a, b], [1.0, 1.0])
    bs = orc.Basis([[0, 0, 0], [0, R, 0]], [0, 1], [0, 0], [1, 1], [0, 1], [a, b], cf)
    v = orc.eri_block(bs, 0, 0, 1, 1)[0, 0, 0, 0]
    rho = 2 * a * 2 * b / (2 * a + 2 * b)
    assert v == pytest.approx(float(mp.erf(mp.sqrt(rho) * R) / R), rel=1e-13)
    assert v == pytest.approx(g["value"], rel=1e-13)


# ---------------------------------------------------------------- P5 contraction + normalisation
def p5_basis(orc):
    g = GOLD["P5"]
    e, c = g["exponents"], g["coefficients"]
    sl, sn, so = [0, 0], [3, 3], [0, 3]
    cf = orc.normalize(sl, sn, so, e + e, c + c)
    return orc.Basis([[0, 0, 0], [0, 0, g["R"]]], [0, 1], sl, sn, so, e + e, cf)


def test_p5_contracted(orc):
    g = GOLD["P5"]
    G = orc.eri_tensor(p5_basis(orc))
    assert G[0, 0, 0, 0] == pytest.approx(g["1111"], abs=2e-10)
    assert G[0, 0, 1, 1] == pytest.approx(g["1122"], abs=2e-10)
    assert G[1, 0, 0, 0] == pytest.approx(g["2111"], abs=2e-10)
    assert G[1, 0, 1, 0] == pytest.approx(g["2121"], abs=2e-10)
    # and live, from the s-type closed form summed over primitives (contraction pin)
    bs = p5_basis(orc)
    ref = mp.mpf(0)
    cen = [bs.xyz[0], bs.xyz[1]]
    for i, j, k, l in itertools.product(range(3), repeat=4):
        ref += (bs.coef[3 + i] * bs.coef[j] * bs.coef[3 + k] * bs.coef[l]
                * ssss_closed(bs.expo[3 + i], bs.expo[j], bs.expo[3 + k], bs.expo[l], cen[1], cen[0], cen[1], cen[0]))
    assert G[1, 0, 1, 0] == pytest.approx(float(ref), rel=1e-13)


@pytest.mark.parametrize("L", [0, 1, 2, 3])
def test_normaliser_unit_self_overlap(orc, L):
    """(L,0,0) component has unit self-overlap; overlap evaluated by numerical quadrature (mpmath)."""
    rng = np.random.default_rng(40 + L)
    n = 4
    e = np.exp(rng.uniform(np.log(0.1), np.log(100), size=n))
    c = rng.uniform(0.1, 1, size=n)
    d = orc.normalize([L], [n], [0], e, c)
    S = mp.mpf(0)
    for i in range(n):
        for j in range(n):
            p = mp.mpf(e[i]) + mp.mpf(e[j])
            ix = mp.quad(lambda x: x ** (2 * L) * mp.exp(-p * x * x), [-mp.inf, 0, mp.inf])
            iy = mp.quad(lambda x: mp.exp(-p * x * x), [-mp.inf, 0, mp.inf])
            S += d[i] * d[j] * ix * iy * iy
    assert float(S) == pytest.approx(1.0, rel=1e-13)


# ---------------------------------------------------------------- P6 one-centre, high L, independent of OS
def p6_ref(i, j, k, zeta, eta):
    if i % 2 or j % 2 or k % 2:
        return 0.0
    n = i + j + k
    ang = mp.fac2(i - 1) * mp.fac2(j - 1) * mp.fac2(k - 1) / mp.fac2(n + 1)
    rad = mp.quad(lambda r: r ** (n + 1) * mp.exp(-zeta * r * r) * mp.erf(mp.sqrt(eta) * r), [0, 2, 6, mp.inf])
    return float(4 * mp.pi * ang * (mp.pi / eta) ** 1.5 * rad)


def test_p6_golden_and_quadrature(orc):
    g = GOLD["P6"]
    zeta, eta = g["zeta"], g["eta"]
    for (i, j, k), val in g["values"]:
        assert p6_ref(i, j, k, mp.mpf(zeta), mp.mpf(eta)) == pytest.approx(val, rel=1e-12, abs=1e-15)
    for (i, j, k), val in g["zeta_eta_2"]:
        assert p6_ref(i, j, k, mp.mpf(2), mp.mpf(2)) == pytest.approx(val, rel=1e-12)


@pytest.mark.parametrize("side", ["bra", "ket"])
@pytest.mark.parametrize("la,lb", [(0, 0), (1, 1), (2, 0), (2, 2), (3, 1), (3, 2), (3, 3), (1, 3)])
def test_p6_one_centre_products(orc, side, la, lb):
    """All four primitives on one centre: (a b|ss) depends only on the product powers; exercises the
    VRR to degree la+lb and the HRR with A = B.  By bra<->ket symmetry the same numbers pin the ket VRR."""
    zeta, eta = 1.3, 0.9
    za = 0.4
    specs = [(0, la, za), (0, lb, zeta - za), (0, 0, 0.25), (0, 0, eta - 0.25)]
    bs = prim_basis(orc, [[0.3, -0.2, 0.7]], specs)
    blk = orc.eri_block(bs, 0, 1, 2, 3)[:, :, 0, 0] if side == "bra" else orc.eri_block(bs, 2, 3, 0, 1)[0, 0, :, :]
    for ia, a in enumerate(comps(la)):
        for ib, b in enumerate(comps(lb)):
            ref = p6_ref(a[0] + b[0], a[1] + b[1], a[2] + b[2], mp.mpf(zeta), mp.mpf(eta))
            assert blk[ia, ib] == pytest.approx(ref, rel=2e-12, abs=1e-14), (a, b)


# ---------------------------------------------------------------- P7 derivative identity (multi-centre, all slots)
def _block_slot(orc, centers, ls, zs, slot, dl):
    """Primitive block with angular momentum of `slot` changed by dl; returns array indexed by components."""
    l2 = list(ls)
    l2[slot] += dl
    bs = prim_basis(orc, centers, [(i, l2[i], zs[i]) for i in range(4)])
    return orc.eri_block(bs, 0, 1, 2, 3)


@pytest.mark.parametrize("slot", [0, 1, 2, 3])
@pytest.mark.parametrize("ls", [(0, 0, 0, 0), (1, 0, 1, 0), (1, 1, 0, 1), (2, 1, 1, 0), (2, 2, 1, 1), (2, 0, 2, 2)])
def test_p7_derivative_identity(orc, slot, ls):
    """(.., a+1_i, ..) = [ d/dA_i (.., a, ..) + a_i (.., a-1_i, ..) ] / (2 alpha) for unnormalised primitives."""
    rng = np.random.default_rng(100 + slot)
    centers = rng.normal(0, 0.8, size=(4, 3))
    zs = np.exp(rng.uniform(np.log(0.3), np.log(3.0), size=4))
    l = ls[slot]
    up = _block_slot(orc, centers, ls, zs, slot, +1)
    dn = _block_slot(orc, centers, ls, zs, slot, -1) if l > 0 else None
    h = 2e-3
    for i in range(3):
        def at(shift):
            c2 = centers.copy(); c2[slot, i] += shift
            return _block_slot(orc, c2, ls, zs, slot, 0)
        deriv = (-at(2 * h) + 8 * at(h) - 8 * at(-h) + at(-2 * h)) / (12 * h)
        for ic, c in enumerate(comps(l)):
            cu = list(c); cu[i] += 1
            iu = comps(l + 1).index(tuple(cu))
            sel = [slice(None)] * 4
            sel_u = list(sel); sel_u[slot] = iu
            sel_c = list(sel); sel_c[slot] = ic
            rhs = deriv[tuple(sel_c)].copy()
            if c[i] > 0:
                cd = list(c); cd[i] -= 1
                idn = comps(l - 1).index(tuple(cd))
                sel_d = list(sel); sel_d[slot] = idn
                rhs = rhs + c[i] * dn[tuple(sel_d)]
            rhs = rhs / (2 * zs[slot])
            lhs = up[tuple(sel_u)]
            scale = max(1e-3, np.abs(lhs).max())
            assert np.abs(lhs - rhs).max() <= 2e-8 * scale + 1e-10


@pytest.mark.parametrize("ls", [(3, 3, 3, 3), (3, 2, 3, 1), (3, 0, 2, 3)])
def test_p7_derivative_identity_high_l(orc, ls):
    """Same identity at f level on slot 0 and slot 3 (where the class sweep of the GPU path needs it most)."""
    for slot in (0, 3):
        ls2 = list(ls); ls2[slot] = 2        # raises d -> f
        test_p7_derivative_identity(orc, slot, tuple(ls2))


# ---------------------------------------------------------------- P8 axis permutations / reflections
def _general_block(orc, centers, ls, rng):
    specs = []
    nprim = 2
    exps, coefs, off = [], [], []
    for i in range(4):
        off.append(len(exps))
        exps += list(np.exp(rng.uniform(np.log(0.2), np.log(5.0), size=nprim)))
        coefs += list(rng.uniform(0.2, 1.0, size=nprim))
    return lambda cen: orc.eri_block(orc.Basis(cen, [0, 1, 2, 3], list(ls), [nprim] * 4, off, exps, coefs), 0, 1, 2, 3)


@pytest.mark.parametrize("ls", [(1, 0, 0, 0), (1, 1, 1, 1), (2, 1, 0, 1), (2, 2, 2, 2), (3, 1, 2, 0), (3, 3, 3, 3),
                                (0, 3, 1, 2)])
def test_p8_axis_permutation_and_reflection(orc, ls):
    rng = np.random.default_rng(8)
    centers = rng.normal(0, 1.0, size=(4, 3))
    f = _general_block(orc, centers, ls, rng)
    base = f(centers)
    cs = [comps(l) for l in ls]
    for perm in [(1, 2, 0), (2, 0, 1), (1, 0, 2), (0, 2, 1)]:
        # new coordinates r'_k = r_perm[k]; a function with powers p in old axes has powers p'_k = p_perm[k]
        got = f(centers[:, list(perm)])
        idx = [[cs[s].index(tuple(c[perm[k]] for k in range(3))) for c in cs[s]] for s in range(4)]
        mapped = got[np.ix_(*idx)]
        np.testing.assert_allclose(mapped, base, rtol=1e-11, atol=2e-13 * max(1.0, np.abs(base).max()))
    for ax in range(3):
        refl = centers.copy(); refl[:, ax] *= -1
        got = f(refl)
        sign = np.ones_like(base)
        for s in range(4):
            sg = np.array([(-1.0) ** c[ax] for c in cs[s]])
            shape = [1] * 4; shape[s] = len(sg)
            sign = sign * sg.reshape(shape)
        np.testing.assert_allclose(got * sign, base, rtol=1e-11, atol=2e-13 * max(1.0, np.abs(base).max()))


# ---------------------------------------------------------------- P9 / P10 / P13 on small workloads
@pytest.mark.parametrize("cfg", [0, "0b"])
def test_p9_p10_tensor_symmetry_and_schwarz(orc, cfg):
    w = W.make(cfg)
    bs = orc.basis_from_workload(w)
    G = orc.eri_tensor(bs)
    for p in [(1, 0, 2, 3), (0, 1, 3, 2), (2, 3, 0, 1), (3, 2, 1, 0), (1, 0, 3, 2), (2, 3, 1, 0), (3, 2, 0, 1)]:
        np.testing.assert_allclose(G.transpose(p), G, rtol=0, atol=1e-13 * np.abs(G).max())
    N = bs.nbf
    diag = np.einsum("ijij->ij", G)
    assert diag.min() >= -1e-15
    # |(mn|ls)| <= sqrt((mn|mn)) sqrt((ls|ls)) elementwise, and <= Q_AB Q_CD shellwise
    bound = np.sqrt(np.abs(diag))
    assert (np.abs(G) <= bound[:, :, None, None] * bound[None, None, :, :] * (1 + 1e-12) + 1e-15).all()
    Q = orc.schwarz(bs)
    o = bs.bf_off
    for A in range(bs.nshells):
        for B in range(bs.nshells):
            blkmax = np.sqrt(np.abs(diag[o[A]:o[A + 1], o[B]:o[B + 1]]).max())
            assert Q[A, B] == pytest.approx(blkmax, rel=1e-13)
    # the ERI supermatrix is positive semidefinite
    ev = np.linalg.eigvalsh(G.reshape(N * N, N * N))
    assert ev.min() >= -1e-10 * ev.max()


def test_p13_long_double_agreement(orc):
    w = W.make(1)
    bs = orc.basis_from_workload(w)
    rng = np.random.default_rng(13)
    worst = 0.0
    for _ in range(60):
        A, B, C, D = rng.integers(0, bs.nshells, size=4)
        d = orc.eri_block(bs, A, B, C, D)
        ld = orc.eri_block(bs, A, B, C, D, long_double=True)
        scale = max(np.abs(d).max(), 1e-8)
        worst = max(worst, float(np.abs(d - ld.astype(np.float64)).max() / scale))
        assert np.abs(ld - d).max() <= 1e-13 * scale + 1e-15   # absolute floor: integrals are O(1)
    # highest class too
    w3 = W.make_custom(np.random.default_rng(3).normal(0, 1.2, (4, 3)), [(0, 3), (1, 3), (2, 3), (3, 3)], seed=77)
    b3 = orc.basis_from_workload(w3)
    d = orc.eri_block(b3, 0, 1, 2, 3); ld = orc.eri_block(b3, 0, 1, 2, 3, long_double=True)
    assert np.abs(ld - d).max() <= 1e-12 * np.abs(d).max()


def test_p13_documented_hrr_cancellation_case(orc):
    """DESIGN.md R-19 / R-22: cfg 1 shells (35, 23) -- a diffuse p shell 8.5 bohr from a tight d shell.  Before R-22 the
    single-orientation fp64 core lost digits there (the HRR shifted angular momentum onto the tight shell); with the
    recurrences built on the centre nearest to each primitive pair's product centre neither core depends on the order the
    two shells are given in, and the Schwarz table (long-double core) matches the block's largest diagonal element."""
    w = W.make(1)
    bs = orc.basis_from_workload(w)
    A, B = 35, 23
    ld1 = orc.eri_block(bs, A, B, A, B, long_double=True)
    ld2 = orc.eri_block(bs, B, A, B, A, long_double=True).transpose(1, 0, 3, 2)
    scale = float(np.abs(ld1).max())
    assert float(np.abs(ld1 - ld2).max()) <= 1e-14                  # order-independent to 1e-14 absolute in long double
    assert scale < 1e-6
    d1 = orc.eri_block(bs, A, B, A, B)
    assert float(np.abs(d1 - ld1.astype(np.float64)).max()) <= 1e-10  # fp64 core: absolute error stays tiny ...
    Q = orc.schwarz(bs)
    diag = max(float(abs(ld1[i, j, i, j])) for i in range(ld1.shape[0]) for j in range(ld1.shape[1]))
    assert Q[A, B] == pytest.approx(np.sqrt(diag), rel=1e-13)         # ... and the Schwarz table uses the ld core


@pytest.mark.parametrize("ls", [(1, 3), (3, 3), (0, 3), (2, 3), (3, 1)])
def test_p15_recurrence_centre_order_independence(orc, ls):
    """DESIGN.md R-22: every primitive quartet is evaluated with the recurrences built on the centre nearest to its
    Gaussian product centre, so the identity (ab|cd) = (ba|cd) = (ab|dc) = (ba|dc) of the definition
    must hold to rounding whichever order the shells are handed over in -- also in plain fp64, also for the case that
    broke the single-orientation core: a very tight high-l shell 11 bohr from a shell with a diffuse primitive
    (cfg 3 shells (242, 294): relative error 33% on Q in long double before R-22).  A wrong index permutation when the
    four orientation groups are added, or a primitive pair left out of every group, fails this test.  (A tie alpha == beta
    counted in BOTH groups is order-symmetric and would pass here: that mistake is caught by P5, whose two shells carry
    the same exponent set and whose golden values a double-counted tie changes, and by P16's mpmath values.)"""
    atoms = np.array([[0.0, 0.0, 0.0], [6.3, -7.1, 5.4], [0.4, 1.1, -0.3], [5.9, -6.5, 5.0]])
    la, lb = ls
    exps = {0: [4595.251], 1: [38.639, 0.05, 376.079], 2: [2019.87, 0.246, 4.992], 3: [1.7, 0.3]}
    cofs = {0: [0.75], 1: [1.0, 0.77, 0.34], 2: [0.53, 0.22, 0.17], 3: [0.6, 0.4]}
    lsh = [lb, la, la, lb]            # shell 0 (tight, single primitive) carries lb; shell 1 (mixed) carries la
    s_np = np.array([len(exps[i]) for i in range(4)], np.int32)
    s_off = np.concatenate([[0], np.cumsum(s_np)[:-1]]).astype(np.int32)
    e = np.array(sum((exps[i] for i in range(4)), []), np.float64)
    c = np.array(sum((cofs[i] for i in range(4)), []), np.float64)
    nbf = sum((l + 1) * (l + 2) // 2 for l in lsh)
    w = W.Workload("p15", atoms, np.arange(4, dtype=np.int32), np.array(lsh, np.int32), s_np, s_off, e, c,
                   np.eye(nbf), 0.0)
    bs = orc.basis_from_workload(w)
    for ld in (False, True):
        ref = orc.eri_block(bs, 0, 1, 2, 3, long_double=ld).astype(np.float64)
        scale = float(np.abs(ref).max())
        assert scale > 0
        for perm, tr in (((1, 0, 2, 3), (1, 0, 2, 3)), ((0, 1, 3, 2), (0, 1, 3, 2)), ((1, 0, 3, 2), (1, 0, 3, 2))):
            sh = [0, 1, 2, 3]
            other = orc.eri_block(bs, *[sh[p] for p in perm], long_double=ld).astype(np.float64).transpose(tr)
            assert float(np.abs(other - ref).max()) <= 2e-13 * scale
    # fp64 and long double agree: nothing left for extra precision to repair
    d = orc.eri_block(bs, 0, 1, 2, 3); l_ = orc.eri_block(bs, 0, 1, 2, 3, long_double=True).astype(np.float64)
    assert float(np.abs(d - l_).max()) <= 2e-13 * float(np.abs(l_).max())
    # the pair that exposed it: diagonal block in both orders
    for (A, B) in ((0, 1),):
        b1 = orc.eri_block(bs, A, B, A, B); b2 = orc.eri_block(bs, B, A, B, A).transpose(1, 0, 3, 2)
        assert float(np.abs(b1 - b2).max()) <= 2e-13 * float(np.abs(b1).max())


@pytest.mark.parametrize("ls", [(3, 2, 3, 1), (3, 3, 3, 3), (2, 2, 2, 1)])
def test_p9_eightfold_symmetry_d_and_f(orc, ls):
    """P9 at d and f level on four distinct centres: the eight index permutations of (ab|cd) evaluated as eight
    separate shell quartets (each with its own recurrence centres and HRR direction) agree to 1e-13 of the block's
    largest element, in the fp64 core and in the long double core.  Exponents span tight and diffuse."""
    atoms = np.array([[0.0, 0.1, -0.2], [2.9, -1.4, 0.5], [-0.6, 3.1, 1.9], [1.7, 2.8, -3.2]])
    w = W.make_custom(atoms, [(i, ls[i]) for i in range(4)], seed=909 + sum(ls), emin=0.05, emax=500.0, nprim=4)
    bs = orc.basis_from_workload(w)
    for ld in (False, True):
        ref = orc.eri_block(bs, 0, 1, 2, 3, long_double=ld).astype(np.float64)
        scale = float(np.abs(ref).max())
        assert scale > 1e-12
        # (shells handed over, axes that bring the result back to [a, b, c, d] order)
        perms = [((1, 0, 2, 3), (1, 0, 2, 3)), ((0, 1, 3, 2), (0, 1, 3, 2)), ((1, 0, 3, 2), (1, 0, 3, 2)),
                 ((2, 3, 0, 1), (2, 3, 0, 1)), ((3, 2, 0, 1), (3, 2, 0, 1)), ((2, 3, 1, 0), (2, 3, 1, 0)),
                 ((3, 2, 1, 0), (3, 2, 1, 0))]
        for sh, _ in perms:
            other = orc.eri_block(bs, *sh, long_double=ld).astype(np.float64)
            # other[i_sh0, i_sh1, i_sh2, i_sh3]: move axis k (shell sh[k]) to position sh[k]
            back = np.moveaxis(other, [0, 1, 2, 3], list(sh))
            assert back.shape == ref.shape
            assert float(np.abs(back - ref).max()) <= 1e-13 * scale, (sh, ld)
