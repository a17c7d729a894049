"""Pin P16: the oracle's high-L multi-centre integrals against an evaluation that shares nothing with it.

The oracle computes (ab|cd) by Obara-Saika/HGP recurrences with the recurrence centre chosen per primitive pair
(R-22).  What showed that those values are right was internal consistency only (two orders agree, fp64 =
long double).  Here the same integrals are evaluated by a different algorithm in 50-digit arithmetic, written out in
this file: the McMurchie-Davidson expansion of each Gaussian product in Hermite Gaussians,

    (ab|cd) = 2 pi^(5/2) / (p q sqrt(p+q)) sum_{tuv} E^{ab}_{tuv} sum_{t'u'v'} (-1)^{t'+u'+v'} E^{cd}_{t'u'v'}
              R_{t+t', u+u', v+v'}(alpha, P - Q),           alpha = p q / (p+q),
    E^{i+1,j}_t = E^{ij}_{t-1}/(2p) + X_PA E^{ij}_t + (t+1) E^{ij}_{t+1},   E^{00}_0 = exp(-a b X_AB^2 / p)   (per axis),
    R^n_{000} = (-2 alpha)^n F_n(alpha |PQ|^2),   R^n_{t+1,u,v} = t R^{n+1}_{t-1,u,v} + X_PQ R^{n+1}_{t,u,v},

with the Boys function from mpmath's incomplete gamma function.  The MD code itself is first checked against the
survey's closed forms (P4 two-centre s, P6 one-centre f), then the oracle must reproduce it to 1e-12 of the block's
largest element and to 1e-11 relative element by element where the element is not negligible (fp64 core; 1e-15 and
1e-14 for the long double core the Schwarz table and J/K use) for
  (1) a single primitive quartet at f level with the exponent mix that broke the first oracle (4595 next to 0.05,
      11 bohr apart), in all four classes (fp|df), (pf|fd), (ff|ff), (fd|pf);
  (2) a contracted quartet with tight and diffuse primitives on every shell.
"""
import functools
import itertools
import json
import os

import mpmath as mp
import numpy as np
import pytest

from paper_2406_11185_b200 import workloads as W

mp.mp.dps = 50
GOLD = json.load(open(os.path.join(os.path.dirname(__file__), "golden", "survey_pins.json")))


def comps(l):
    return [(x, y, l - x - y) for x in range(l, -1, -1) for y in range(l - x, -1, -1)]


def boys_mp(n, T):
    T = mp.mpf(T)
    if T == 0:
        return mp.mpf(1) / (2 * n + 1)
    return mp.gammainc(n + mp.mpf(1) / 2, 0, T) / (2 * T ** (n + mp.mpf(1) / 2))


def hermite_E(i, j, a, b, XA, XB):
    """E^{ij}_t, t = 0..i+j, one axis; XA, XB = coordinates of the two centres on that axis."""
    p = a + b
    XP = (a * XA + b * XB) / p
    XPA, XPB = XP - XA, XP - XB
    E = {(0, 0): [mp.e ** (-a * b / p * (XA - XB) ** 2)]}

    def get(tab, t):
        return tab[t] if 0 <= t < len(tab) else mp.mpf(0)
    for ii in range(i):
        prev = E[(ii, 0)]
        E[(ii + 1, 0)] = [get(prev, t - 1) / (2 * p) + XPA * get(prev, t) + (t + 1) * get(prev, t + 1)
                          for t in range(ii + 2)]
    for jj in range(j):
        for ii in range(i + 1):
            prev = E[(ii, jj)]
            E[(ii, jj + 1)] = [get(prev, t - 1) / (2 * p) + XPB * get(prev, t) + (t + 1) * get(prev, t + 1)
                               for t in range(ii + jj + 2)]
    return E[(i, j)]


def hermite_R(L, alpha, PQ):
    """R^0_{tuv} for t+u+v <= L."""
    T = alpha * sum(x * x for x in PQ)
    F = [boys_mp(n, T) for n in range(L + 1)]

    @functools.lru_cache(maxsize=None)
    def R(n, t, u, v):
        if t < 0 or u < 0 or v < 0:
            return mp.mpf(0)
        if t == u == v == 0:
            return (-2 * alpha) ** n * F[n]
        if t > 0:
            return (t - 1) * R(n + 1, t - 2, u, v) + PQ[0] * R(n + 1, t - 1, u, v)
        if u > 0:
            return (u - 1) * R(n + 1, t, u - 2, v) + PQ[1] * R(n + 1, t, u - 1, v)
        return (v - 1) * R(n + 1, t, u, v - 2) + PQ[2] * R(n + 1, t, u, v - 1)
    return R


def md_primitive(a, A, la, b, B, lb, c, C, lc, d, D, ld, which):
    """Unnormalised primitive integrals (a_comp b_comp | c_comp d_comp) for the component tuples in `which`."""
    a, b, c, d = (mp.mpf(x) for x in (a, b, c, d))
    A, B, C, D = ([mp.mpf(float(x)) for x in v] for v in (A, B, C, D))
    p, q = a + b, c + d
    P = [(a * A[i] + b * B[i]) / p for i in range(3)]
    Qc = [(c * C[i] + d * D[i]) / q for i in range(3)]
    alpha = p * q / (p + q)
    R = hermite_R(la + lb + lc + ld, alpha, [P[i] - Qc[i] for i in range(3)])
    pref = 2 * mp.pi ** (mp.mpf(5) / 2) / (p * q * mp.sqrt(p + q))
    out = {}
    for (ca, cb, cc_, cd) in which:
        Eab = [hermite_E(ca[i], cb[i], a, b, A[i], B[i]) for i in range(3)]
        Ecd = [hermite_E(cc_[i], cd[i], c, d, C[i], D[i]) for i in range(3)]
        s = mp.mpf(0)
        for t, u, v in itertools.product(range(len(Eab[0])), range(len(Eab[1])), range(len(Eab[2]))):
            eab = Eab[0][t] * Eab[1][u] * Eab[2][v]
            for t2, u2, v2 in itertools.product(range(len(Ecd[0])), range(len(Ecd[1])), range(len(Ecd[2]))):
                s += eab * (-1) ** (t2 + u2 + v2) * Ecd[0][t2] * Ecd[1][u2] * Ecd[2][v2] * R(0, t + t2, u + u2, v + v2)
        out[(ca, cb, cc_, cd)] = pref * s
    return out


def test_md_code_against_closed_forms():
    """The mpmath MD evaluation is itself pinned: survey pin P4 (two-centre s, erf closed form) and P6 (one-centre
    f-level closed form), so that P16 compares the oracle with something known to be right."""
    g = GOLD["P4"]
    a, b, R = g["a"], g["b"], g["R"]
    na = (2 * mp.mpf(a) / mp.pi) ** (mp.mpf(3) / 4); nb = (2 * mp.mpf(b) / mp.pi) ** (mp.mpf(3) / 4)
    z = (0, 0, 0)
    v = md_primitive(a, [0, 0, 0], 0, a, [0, 0, 0], 0, b, [0, 0, R], 0, b, [0, 0, R], 0, [(z, z, z, z)])[(z, z, z, z)]
    assert abs(float(v * na * na * nb * nb) - g["value"]) < 1e-15
    rho = (2 * mp.mpf(a)) * (2 * mp.mpf(b)) / (2 * mp.mpf(a) + 2 * mp.mpf(b))
    assert abs(v * na * na * nb * nb - mp.erf(mp.sqrt(rho) * mp.mpf(R)) / mp.mpf(R)) < mp.mpf(10) ** -40
    # P6: (f_xxx f_xxx | s s) on one centre with zeta = 1.3, eta = 0.9 -> 11.72657513937246
    f = (3, 0, 0)
    v = md_primitive(0.5, [0.3, -0.2, 0.1], 3, 0.8, [0.3, -0.2, 0.1], 3, 0.4, [0.3, -0.2, 0.1], 0, 0.5, [0.3, -0.2, 0.1], 0,
                     [(f, f, z, z)])[(f, f, z, z)]
    want = [x[1] for x in GOLD["P6"]["values"] if tuple(x[0]) == (6, 0, 0)][0]
    assert abs(float(v) - want) < 1e-12


def _system(ls, exps, cofs, atoms):
    s_np = np.array([len(e) for e in exps], np.int32)
    s_off = np.concatenate([[0], np.cumsum(s_np)[:-1]]).astype(np.int32)
    e = np.array(sum(exps, []), np.float64); c = np.array(sum(cofs, []), np.float64)
    return atoms, np.arange(4, dtype=np.int32), np.array(ls, np.int32), s_np, s_off, e, c


ATOMS = np.array([[0.0, 0.0, 0.0], [6.3, -7.1, 5.4], [0.4, 1.1, -0.3], [5.9, -6.5, 5.0]])       # |A-B| = 10.9 bohr


def _compare(orc, ls, exps, cofs, nsample, seed):
    atoms, s_atom, s_l, s_np, s_off, e, c = _system(ls, exps, cofs, ATOMS)
    bs = orc.Basis(atoms, s_atom, s_l, s_np, s_off, e, c)          # coefficients passed as FINAL: no normalisation
    cA, cB, cC, cD = (comps(l) for l in ls)
    every = list(itertools.product(range(len(cA)), range(len(cB)), range(len(cC)), range(len(cD))))
    rng = np.random.default_rng(seed)
    pick = [every[i] for i in rng.choice(len(every), size=min(nsample, len(every)), replace=False)]
    which = [(cA[i], cB[j], cC[k], cD[m]) for (i, j, k, m) in pick]
    ref = {w_: mp.mpf(0) for w_ in which}
    for ia, ib, ic, id_ in itertools.product(*(range(len(x)) for x in exps)):
        part = md_primitive(exps[0][ia], atoms[0], ls[0], exps[1][ib], atoms[1], ls[1], exps[2][ic], atoms[2], ls[2],
                            exps[3][id_], atoms[3], ls[3], which)
        cf = mp.mpf(cofs[0][ia]) * mp.mpf(cofs[1][ib]) * mp.mpf(cofs[2][ic]) * mp.mpf(cofs[3][id_])
        for w_ in which:
            ref[w_] += cf * part[w_]
    out = {}
    for ld in (False, True):
        blk = orc.eri_block(bs, 0, 1, 2, 3, long_double=ld)
        scale = float(np.abs(np.asarray(blk, np.float64)).max())
        worst_abs = worst_rel = 0.0
        for (i, j, k, m), w_ in zip(pick, which):
            got = mp.mpf(float(blk[i, j, k, m])) if not ld else mp.mpf(str(np.format_float_scientific(blk[i, j, k, m], precision=22)))
            err = abs(got - ref[w_])
            worst_abs = max(worst_abs, float(err) / scale)
            if abs(ref[w_]) > 1e-4 * scale:
                worst_rel = max(worst_rel, float(err / abs(ref[w_])))
        out[ld] = (worst_abs, worst_rel, scale)
    return out


@pytest.mark.parametrize("ls", [(3, 1, 2, 3), (1, 3, 3, 2), (3, 3, 3, 3), (3, 2, 1, 3)])
def test_p16_primitive_quartet_f_level_tight_diffuse(orc, ls):
    """One primitive per shell: alpha = 4595.251 on A, 0.05 on B (10.9 bohr away), 2019.87 on C, 0.3 on D."""
    res = _compare(orc, ls, [[4595.251], [0.05], [2019.87], [0.3]], [[1.0], [1.0], [1.0], [1.0]], nsample=24, seed=16)
    for ld, (wabs, wrel, scale) in res.items():          # measured: fp64 core 3e-14 / 5e-13, long double 2e-17 / 5e-16
        assert scale > 0
        assert wabs <= (1e-15 if ld else 1e-12), (ld, wabs, wrel)
        assert wrel <= (1e-14 if ld else 1e-11), (ld, wabs, wrel)


@pytest.mark.parametrize("ls", [(3, 1, 2, 3), (1, 3, 3, 1), (3, 3, 2, 2)])
def test_p16_contracted_quartet_f_level_tight_diffuse(orc, ls):
    """Contracted shells with the P15 exponent mix (tight and diffuse primitives on the same shell)."""
    exps = [[4595.251, 3.1], [38.639, 0.05, 376.079], [2019.87, 0.246], [1.7, 0.3]]
    cofs = [[0.75, 0.4], [1.0, 0.77, 0.34], [0.53, 0.22], [0.6, 0.4]]
    res = _compare(orc, ls, exps, cofs, nsample=12, seed=17)
    for ld, (wabs, wrel, scale) in res.items():          # measured: fp64 core 2e-15 / 8e-15, long double 1e-18 / 2e-18
        assert wabs <= (1e-15 if ld else 1e-12), (ld, wabs, wrel)
        assert wrel <= (1e-14 if ld else 1e-11), (ld, wabs, wrel)
