"""CPU check of the product's ERI code generator: the recurrence DAGs it emits as CUDA are evaluated in
Python and compared with the oracle, class by class (catches generator mistakes before any GPU time)."""
import math
import os
import sys

import numpy as np
import pytest
from scipy.special import hyp1f1

sys.path.insert(0, os.path.join(os.path.dirname(__file__), "..", "paper_2406_11185_b200", "csrc", "gen"))
import gen_eri  # noqa: E402


def prim_ctx(za, zb, zc, zd, A, B, C, D, L):
    zeta, eta = za + zb, zc + zd
    P = (za * A + zb * B) / zeta
    Q = (zc * C + zd * D) / eta
    W = (zeta * P + eta * Q) / (zeta + eta)
    rho = zeta * eta / (zeta + eta)
    T = rho * np.dot(P - Q, P - Q)
    pref = (2 * math.pi ** 2.5 / (zeta * eta * math.sqrt(zeta + eta))
            * math.exp(-za * zb / zeta * np.dot(A - B, A - B)) * math.exp(-zc * zd / eta * np.dot(C - D, C - D)))
    F = [pref * float(hyp1f1(m + 0.5, m + 1.5, -T)) / (2 * m + 1) for m in range(L + 1)]
    return dict(PA=P - A, WP=W - P, QC=Q - C, WQ=W - Q, inv2z=0.5 / zeta, inv2e=0.5 / eta,
                inv2ze=0.5 / (zeta + eta), roz=rho / zeta, roe=rho / eta, F=F)


CLASSES = [c for c in gen_eri.all_classes(3) if sum(c) <= 8] + [(3, 3, 3, 3), (3, 2, 3, 1)]


@pytest.mark.parametrize("cls", CLASSES, ids=lambda c: "".join("spdf"[x] for x in c))
def test_generated_dag_matches_oracle(orc, cls):
    la, lb, lc, ld = cls
    rng = np.random.default_rng(sum(x * 7 ** i for i, x in enumerate(cls)))
    cen = rng.normal(0, 0.9, size=(4, 3))
    z = np.exp(rng.uniform(np.log(0.3), np.log(4.0), size=4))
    bs = orc.Basis(cen, [0, 1, 2, 3], list(cls), [1] * 4, [0, 1, 2, 3], z, [1.0] * 4)
    ref = orc.eri_block(bs, 0, 1, 2, 3)
    vrr = gen_eri.best_vrr(la, lb, lc, ld)
    hrr = gen_eri.HrrDag(la, lb, lc, ld)
    ctx = prim_ctx(*z, *cen, la + lb + lc + ld)
    acc = vrr.evaluate(ctx)
    got = hrr.evaluate(acc, cen[0] - cen[1], cen[2] - cen[3])
    scale = np.abs(ref).max()
    for (ia, ib, ic, idd), v in got.items():
        assert abs(v - ref[ia, ib, ic, idd]) <= 2e-12 * scale
    assert len(got) == ref.size
    if (la, lb) == (lc, ld):
        diag = gen_eri.HrrDag(la, lb, lc, ld, diag_only=True).evaluate(acc, cen[0] - cen[1], cen[2] - cen[3])
        assert len(diag) == ref.shape[0] * ref.shape[1]
        for (ia, ib, ic, idd), v in diag.items():
            assert ia == ic and ib == idd and abs(v - ref[ia, ib, ic, idd]) <= 2e-12 * scale


def test_all_direction_rules_agree():
    cen = np.random.default_rng(1).normal(0, 1, (4, 3)); z = [0.7, 1.1, 0.5, 2.0]
    ctx = prim_ctx(*z, *cen, 6)
    base = None
    for how in ("first", "last", "max", "min"):
        acc = np.array(gen_eri.VrrDag(2, 1, 2, 1, how).evaluate(ctx))
        base = acc if base is None else base
        np.testing.assert_allclose(acc, base, rtol=1e-12, atol=1e-14)
