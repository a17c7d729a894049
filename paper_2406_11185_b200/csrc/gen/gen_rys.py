#!/usr/bin/env python3
"""gen_rys.py -- Rys quadrature tables for the high-L class kernels (csrc/adft_rys.cuh).

For N = 1..NMAX the N-point Rys quadrature at argument T is the Gauss rule of the weight e^{-T t^2} on t in [0,1]
in the variable u = t^2:   sum_i w_i(T) u_i(T)^k = F_k(T) = int_0^1 t^{2k} e^{-T t^2} dt,   k = 0..2N-1
(Dupuis, Rys, King 1976; the method PAPER.md:72 names beside HGP).  Nodes and weights are smooth in T, so they are
tabulated as piecewise Chebyshev polynomials on [0, TMAX) (interval width H, NCOEF coefficients per interval); for
T >= TMAX the weight is Gauss-Hermite to 1e-28 and u_i = x_i^2 / T, w_i = h_i / sqrt(T) with (x_i, h_i) the
positive-half rule of H_{2N}.  Everything is computed with mpmath at DPS digits (moments -> Hankel matrix ->
Cholesky -> Jacobi matrix -> eigen decomposition); nothing here is shared with oracle/.

Blob layout (float64, little endian):
  header[8]: magic 5259531.0, NMAX, TMAX, H, NCOEF, 0, 0, 0
  for N = 1..NMAX: for interval k = 0..TMAX/H-1: for f = 0..2N-1 (u_0..u_{N-1}, w_0..w_{N-1}): NCOEF Chebyshev
      coefficients c_j of  f(T) = sum_j c_j T_j(x),  x = 2 (T - k H)/H - 1     (c_0 is the full constant term)
  for N = 1..NMAX: x_i^2 (N values), h_i (N values) of the asymptotic rule
"""
from __future__ import annotations

import argparse
import multiprocessing as mp_
import struct
import sys

import mpmath as mp

NMAX = 9          # (gg|gg): L = 16, L/2 + 1 = 9 roots
TMAX = 80.0
H = 1.0
NCOEF = 16
DPS = 100
MAGIC = 5259531.0


def boys_moments(T, n):
    """F_k(T), k = 0..n-1, at working precision."""
    T = mp.mpf(T)
    if T == 0:
        return [mp.mpf(1) / (2 * k + 1) for k in range(n)]
    return [mp.gammainc(k + mp.mpf(1) / 2, 0, T) / (2 * T ** (k + mp.mpf(1) / 2)) for k in range(n)]


def gauss_from_moments(m, N):
    """Golub-Welsch from the moments m_0..m_{2N-1}... (needs m_0..m_{2N}); returns nodes, weights."""
    M = mp.matrix(N + 1, N + 1)
    for i in range(N + 1):
        for j in range(N + 1):
            M[i, j] = m[i + j]
    R = mp.cholesky(M).T                      # M = R^T R, R upper triangular
    alpha = [None] * N
    beta = [None] * max(N - 1, 0)
    for j in range(N):
        alpha[j] = R[j, j + 1] / R[j, j] - (R[j - 1, j] / R[j - 1, j - 1] if j > 0 else 0)
    for j in range(N - 1):
        beta[j] = R[j + 1, j + 1] / R[j, j]
    Jm = mp.matrix(N, N)
    for j in range(N):
        Jm[j, j] = alpha[j]
    for j in range(N - 1):
        Jm[j, j + 1] = Jm[j + 1, j] = beta[j]
    E, Q = mp.eigsy(Jm)
    idx = sorted(range(N), key=lambda i: E[i])
    nodes = [E[i] for i in idx]
    weights = [m[0] * Q[0, i] ** 2 for i in idx]
    return nodes, weights


def rys(T, N):
    mp.mp.dps = DPS
    m = boys_moments(T, 2 * N + 1)
    return gauss_from_moments(m, N)


def hermite_half(N):
    """Gauss rule of e^{-x^2} on [0, inf) in u = x^2 restricted to even polynomials: moments
    int_0^inf x^{2k} e^{-x^2} dx = Gamma(k+1/2)/2."""
    mp.mp.dps = DPS
    m = [mp.gamma(k + mp.mpf(1) / 2) / 2 for k in range(2 * N + 1)]
    return gauss_from_moments(m, N)


def cheb_fit_interval(args):
    """Chebyshev coefficients of u_i(T), w_i(T) on [a, a+H): interpolation at the NCOEF Chebyshev points."""
    N, k, ncoef, h = args
    mp.mp.dps = DPS
    a = mp.mpf(k) * h
    xs = [mp.cos(mp.pi * (j + mp.mpf(1) / 2) / ncoef) for j in range(ncoef)]
    vals = []
    for x in xs:
        u, w = rys(a + (x + 1) * h / 2, N)
        vals.append(list(u) + list(w))
    out = []
    for f in range(2 * N):
        c = []
        for j in range(ncoef):
            s = sum(vals[i][f] * mp.cos(mp.pi * j * (i + mp.mpf(1) / 2) / ncoef) for i in range(ncoef))
            c.append(float(s * (1 if j == 0 else 2) / ncoef))
        out.append(c)
    return N, k, out


def eval_table(tab, N, T):
    """Evaluate the tabulated rule (same arithmetic as the device code, in fp64); tab = dict from build_tables."""
    if T >= tab["tmax"]:
        x2, hw = tab["asym"][N]
        return [v / T for v in x2], [v / T ** 0.5 for v in hw]
    k = min(int(T / tab["h"]), int(round(tab["tmax"] / tab["h"])) - 1)
    x = 2.0 * (T - k * tab["h"]) / tab["h"] - 1.0
    res = []
    for c in tab["cheb"][N][k]:
        b1 = b2 = 0.0
        for cj in reversed(c[1:]):               # Clenshaw
            b1, b2 = 2.0 * x * b1 - b2 + cj, b1
        res.append(x * b1 - b2 + c[0])
    return res[:N], res[N:]


def build_tables(nmax=NMAX, tmax=TMAX, h=H, ncoef=NCOEF, procs=None):
    nint = int(round(tmax / h))
    jobs = [(N, k, ncoef, h) for N in range(1, nmax + 1) for k in range(nint)]
    cheb = {N: [None] * nint for N in range(1, nmax + 1)}
    with mp_.Pool(procs) as pool:
        for N, k, out in pool.imap_unordered(cheb_fit_interval, jobs, chunksize=4):
            cheb[N][k] = out
    asym = {}
    for N in range(1, nmax + 1):
        u, w = hermite_half(N)
        asym[N] = ([float(v) for v in u], [float(v) for v in w])
    return {"nmax": nmax, "tmax": tmax, "h": h, "ncoef": ncoef, "cheb": cheb, "asym": asym}


def write_blob(path, tab):
    nint = int(round(tab["tmax"] / tab["h"]))
    vals = [MAGIC, float(tab["nmax"]), tab["tmax"], tab["h"], float(tab["ncoef"]), 0.0, 0.0, 0.0]
    for N in range(1, tab["nmax"] + 1):
        for k in range(nint):
            for c in tab["cheb"][N][k]:
                vals.extend(c)
    for N in range(1, tab["nmax"] + 1):
        vals.extend(tab["asym"][N][0])
        vals.extend(tab["asym"][N][1])
    with open(path, "wb") as f:
        f.write(struct.pack("<%dd" % len(vals), *vals))
    return len(vals)


def read_blob(path):
    raw = open(path, "rb").read()
    v = struct.unpack("<%dd" % (len(raw) // 8), raw)
    assert v[0] == MAGIC
    nmax, tmax, h, ncoef = int(v[1]), v[2], v[3], int(v[4])
    nint = int(round(tmax / h))
    p = 8
    cheb, asym = {}, {}
    for N in range(1, nmax + 1):
        cheb[N] = []
        for k in range(nint):
            fs = []
            for f in range(2 * N):
                fs.append(list(v[p:p + ncoef])); p += ncoef
            cheb[N].append(fs)
    for N in range(1, nmax + 1):
        asym[N] = (list(v[p:p + N]), list(v[p + N:p + 2 * N])); p += 2 * N
    assert p == len(v)
    return {"nmax": nmax, "tmax": tmax, "h": h, "ncoef": ncoef, "cheb": cheb, "asym": asym}


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--out", required=True)
    ap.add_argument("--procs", type=int, default=None)
    ap.add_argument("--check", type=int, default=0, help="random test points per N compared with the exact rule")
    a = ap.parse_args()
    tab = build_tables(procs=a.procs)
    n = write_blob(a.out, tab)
    print(f"wrote {n} doubles to {a.out}")
    if a.check:
        import random
        rnd = random.Random(1)
        tab = read_blob(a.out)
        for N in range(1, NMAX + 1):
            worst = 0.0
            for _ in range(a.check):
                T = rnd.uniform(0, 1.25 * TMAX)
                u, w = eval_table(tab, N, T)
                ue, we = rys(T, N)
                w0 = max(float(x) for x in we)
                for i in range(N):
                    worst = max(worst, abs(u[i] - float(ue[i])) / float(ue[i]), abs(w[i] - float(we[i])) / w0)
            print(f"N={N}: worst rel error of u_i, w_i/max(w): {worst:.2e}")


if __name__ == "__main__":
    sys.exit(main())
