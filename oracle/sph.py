"""ORACLE -- TEST INFRASTRUCTURE ONLY.  Cartesian -> real-solid-harmonic transformation of J and K (SURVEY.md 8(f4)
"spherical-harmonic output"; PAPER.md:44 the basis functions).  Plain numpy, written from the definition:

  * the real regular solid harmonics S_lm, m = -l..l, as polynomials in x, y, z from the textbook recurrences
    (Helgaker, Jorgensen, Olsen, "Molecular Electronic-Structure Theory", eqs. 6.4.70-6.4.73):
        S_00 = 1
        S_{l+1, l+1}  = c_l (x S_ll - (1 - delta_l0) y S_{l,-l})
        S_{l+1,-l-1}  = c_l (y S_ll + (1 - delta_l0) x S_{l,-l}),      c_l = sqrt(2^delta_l0 (2l+1)/(2l+2))
        S_{l+1, m}    = ((2l+1) z S_lm - sqrt((l+m)(l-m)) r^2 S_{l-1,m}) / sqrt((l+m+1)(l-m+1))
  * all Cartesian components of a shell share one radial function (R-1), so their overlap matrix is
        <x^a y^b z^c | x^a' y^b' z^c'> = (a+a'-1)!! (b+b'-1)!! (c+c'-1)!! / (2L-1)!!   (all sums even, else 0)
    for every exponent and contraction; each S_lm column is scaled to unit norm under it.
  * M_sph = T^T M_cart T with T block diagonal over the shells, spherical order m = -l, ..., +l inside a shell.

It shares nothing with the CUDA library, which tabulates the polynomials instead of generating them.
"""
from __future__ import annotations

import math

import numpy as np


def _comps(l):
    return [(x, y, l - x - y) for x in range(l, -1, -1) for y in range(l - x, -1, -1)]      # R-3 order


def _mul(p, mono, c=1.0):
    out = {}
    for (a, b, d), v in p.items():
        k = (a + mono[0], b + mono[1], d + mono[2])
        out[k] = out.get(k, 0.0) + c * v
    return out


def _add(p, q, cq=1.0):
    out = dict(p)
    for k, v in q.items():
        out[k] = out.get(k, 0.0) + cq * v
    return out


def solid_harmonics(lmax):
    """S[l][m] for m in -l..l as {(a, b, c): coefficient} (Racah-normalised regular solid harmonics)."""
    S = {0: {0: {(0, 0, 0): 1.0}}}
    for l in range(lmax):
        nxt = {}
        c = math.sqrt((2.0 if l == 0 else 1.0) * (2 * l + 1) / (2 * l + 2))
        top = _mul(S[l][l], (1, 0, 0))
        bot = _mul(S[l][l], (0, 1, 0))
        if l > 0:
            top = _add(top, _mul(S[l][-l], (0, 1, 0)), -1.0)
            bot = _add(bot, _mul(S[l][-l], (1, 0, 0)), 1.0)
        nxt[l + 1] = {k: c * v for k, v in top.items()}
        nxt[-l - 1] = {k: c * v for k, v in bot.items()}
        for m in range(-l, l + 1):
            p = _mul(S[l][m], (0, 0, 1), 2 * l + 1)
            if l >= 1 and abs(m) <= l - 1:
                f = math.sqrt((l + m) * (l - m))
                q = S[l - 1][m]
                r2q = _add(_add(_mul(q, (2, 0, 0)), _mul(q, (0, 2, 0))), _mul(q, (0, 0, 2)))
                p = _add(p, r2q, -f)
            d = math.sqrt((l + m + 1) * (l - m + 1))
            nxt[m] = {k: v / d for k, v in p.items()}
        S[l + 1] = nxt
    return S


def _dfact(n):
    return 1.0 if n <= 0 else float(np.prod(np.arange(n, 0, -2, dtype=np.float64)))


def cart_overlap(l):
    """Overlap matrix of the Cartesian components of one shell (unit self-overlap of (L,0,0))."""
    cs = _comps(l)
    M = np.zeros((len(cs), len(cs)))
    for i, a in enumerate(cs):
        for j, b in enumerate(cs):
            s = [a[k] + b[k] for k in range(3)]
            if all(v % 2 == 0 for v in s):
                M[i, j] = _dfact(s[0] - 1) * _dfact(s[1] - 1) * _dfact(s[2] - 1) / _dfact(2 * l - 1)
    return M


def shell_transform(l):
    """T_l [ncart(l), 2l+1]: column m+l holds the unit-norm S_lm in the Cartesian components of the shell."""
    S = solid_harmonics(l)[l]
    cs = _comps(l)
    T = np.zeros((len(cs), 2 * l + 1))
    for m in range(-l, l + 1):
        for k, v in S[m].items():
            T[cs.index(k), m + l] = v
    M = cart_overlap(l)
    for c in range(2 * l + 1):
        T[:, c] /= math.sqrt(T[:, c] @ M @ T[:, c])
    return T


def transform_matrix(shell_l):
    """Block-diagonal T [ncart_total, nsph_total] of a basis."""
    ls = [int(x) for x in shell_l]
    nc = sum((l + 1) * (l + 2) // 2 for l in ls)
    nsp = sum(2 * l + 1 for l in ls)
    T = np.zeros((nc, nsp))
    i = j = 0
    for l in ls:
        t = shell_transform(l)
        T[i:i + t.shape[0], j:j + t.shape[1]] = t
        i += t.shape[0]; j += t.shape[1]
    return T


def cart_to_spherical(shell_l, M_cart):
    T = transform_matrix(shell_l)
    return T.T @ np.asarray(M_cart, np.float64) @ T
