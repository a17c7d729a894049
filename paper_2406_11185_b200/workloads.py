"""Seeded synthetic inputs for the J/K build (BASELINE.json `configs`).

This module is the ONLY code shared by the oracle side and the CUDA side.  It holds
none of the method's arithmetic: no normalisation, no integrals, no screening.  It
draws geometry, shell templates, raw exponents / raw contraction coefficients and the
matrix C, and forms D = s * C C^T (a plain matrix product that is *input*, not method).

The paper's own workloads (329 molecules with def2-tzvpp, water clusters, ubiquitin;
PAPER.md:189-191, 220, 279-281) are not available; these configs stand in for them
(contracted Cartesian shells up to f, heavy/light atoms, tau = 1e-12).

Readings of BASELINE.json taken here are SURVEY.md R-14 .. R-18 (listed in DESIGN.md).

RNG: numpy.random.Generator(PCG64(seed)), seed = 2406111850 + cfg index.  Draw order:
(1) geometry, (2) heavy/light choice, (3) per shell in order: nprim, exponents,
coefficients, (4) C row-major.  cfg 2 and cfg 3 share draws (1)-(2) (separate stream).
"""
from __future__ import annotations

import dataclasses
import numpy as np

SEED_BASE = 2406111850

# shell templates: list of angular momenta per atom kind
HEAVY_SPD = [0, 0, 0, 1, 1, 2]
LIGHT_SP = [0, 0, 1]
HEAVY_SPDF = [0, 0, 0, 1, 1, 2, 3]
LIGHT_SPD = [0, 0, 1, 2]


def ncart(l: int) -> int:
    return (l + 1) * (l + 2) // 2


@dataclasses.dataclass
class Workload:
    name: str
    atoms: np.ndarray          # [natoms, 3] float64, bohr
    shell_atom: np.ndarray     # [nshells] int32
    shell_l: np.ndarray        # [nshells] int32
    shell_nprim: np.ndarray    # [nshells] int32
    shell_off: np.ndarray      # [nshells] int32 offset into exponents / coefficients
    exponents: np.ndarray      # [nprim_total] float64
    coefficients: np.ndarray   # [nprim_total] float64, RAW (un-normalised) contraction coefficients
    D: np.ndarray              # [nbf, nbf] float64 symmetric
    tau: float                 # Schwarz threshold

    @property
    def natoms(self) -> int:
        return int(self.atoms.shape[0])

    @property
    def nshells(self) -> int:
        return int(self.shell_l.shape[0])

    @property
    def nbf(self) -> int:
        return int(sum(ncart(int(l)) for l in self.shell_l))

    def shells_struct(self) -> np.ndarray:
        """[nshells, 4] int32 rows {atom, l, nprim, prim_offset} (adft_shell_t layout)."""
        return np.ascontiguousarray(
            np.stack([self.shell_atom, self.shell_l, self.shell_nprim, self.shell_off], axis=1).astype(np.int32))

    def bf_offsets(self) -> np.ndarray:
        off = np.zeros(self.nshells + 1, dtype=np.int64)
        for i, l in enumerate(self.shell_l):
            off[i + 1] = off[i] + ncart(int(l))
        return off


def _draw_shells(rng, atom_kinds, templates, emin, emax, shared=None, nprim_fixed=None):
    """Per shell in order: nprim, exponents (log-uniform), coefficients U[0.1, 1]."""
    s_atom, s_l, s_np, s_off, exps, cofs = [], [], [], [], [], []
    off = 0
    for ia, kind in enumerate(atom_kinds):
        for l in templates[kind]:
            if shared is not None:
                e, c = shared
                n = len(e)
            else:
                n = nprim_fixed if nprim_fixed is not None else int(rng.integers(1, 7))
                e = np.exp(rng.uniform(np.log(emin), np.log(emax), size=n))
                c = rng.uniform(0.1, 1.0, size=n)
            s_atom.append(ia); s_l.append(l); s_np.append(n); s_off.append(off)
            exps.extend(np.asarray(e, dtype=np.float64).tolist())
            cofs.extend(np.asarray(c, dtype=np.float64).tolist())
            off += n
    return (np.array(s_atom, np.int32), np.array(s_l, np.int32), np.array(s_np, np.int32),
            np.array(s_off, np.int32), np.array(exps, np.float64), np.array(cofs, np.float64))


def _density(rng, nbf, nocc, mode):
    C = rng.standard_normal((nbf, nocc))
    # G = C C^T by rank-1 updates in a fixed order with elementwise IEEE multiplies and adds: bit-identical on every
    # machine.  (A BLAS matmul picks its kernel, and with it the summation order, by CPU type; stored oracle results are
    # keyed by the SHA-256 of the inputs and are made on one machine and checked on another.)
    G = np.zeros((nbf, nbf))
    tmp = np.empty((nbf, nbf))
    Ct = np.ascontiguousarray(C.T)
    for k in range(nocc):
        np.multiply.outer(Ct[k], Ct[k], out=tmp)
        G += tmp
    if mode == "cfg0":
        D = 0.2 * G
    elif mode == "over_nocc":
        D = G / float(nocc)
    elif mode == "trace":
        tr = 0.0
        for i in range(nbf):                  # plain sequential sum: np.trace's pairwise blocks are an implementation detail
            tr += float(G[i, i])
        D = G * (float(nocc) / tr)
    else:
        raise ValueError(mode)
    return np.ascontiguousarray(0.5 * (D + D.T))


def _finish(name, rng, atoms, kinds, templates, emin, emax, nocc, dmode, tau, shared=None, nprim_fixed=None):
    sa, sl, sn, so, ex, co = _draw_shells(rng, kinds, templates, emin, emax, shared, nprim_fixed)
    nbf = int(sum(ncart(int(l)) for l in sl))
    D = _density(rng, nbf, nocc, dmode)
    return Workload(name, np.ascontiguousarray(atoms, dtype=np.float64), sa, sl, sn, so, ex, co, D, tau)


def _lattice60(seed):
    """cfg 2/3 geometry + kinds (R-17): 60 of 64 sites of a 4^3 lattice, spacing 3.5, jitter N(0,0.3)."""
    g = np.random.Generator(np.random.PCG64(seed))
    sites = np.array([[i, j, k] for i in range(4) for j in range(4) for k in range(4)], dtype=np.float64) * 3.5
    keep = np.sort(g.permutation(64)[:60])           # listed in lattice order
    atoms = sites[keep] + g.normal(0.0, 0.3, size=(60, 3))
    heavy = set(g.permutation(60)[:20].tolist())
    kinds = ["H" if i in heavy else "L" for i in range(60)]
    return atoms, kinds


def _sphere300(rng):
    """cfg 4 geometry: 300 points uniform in a sphere, density 0.01/bohr^3, min separation 2.0."""
    n = 300
    R = (3.0 * n / (4.0 * np.pi * 0.01)) ** (1.0 / 3.0)
    pts = []
    while len(pts) < n:
        p = rng.uniform(-R, R, size=3)
        if p[0] * p[0] + p[1] * p[1] + p[2] * p[2] > R * R:
            continue
        if all((p[0] - q[0]) ** 2 + (p[1] - q[1]) ** 2 + (p[2] - q[2]) ** 2 >= 4.0 for q in pts):
            pts.append(p)
    return np.array(pts)


_MADE = {}


def make(cfg: int | str) -> Workload:
    """Build config `cfg` in {0, '0b', 1, 2, 3, 4} (BASELINE.json `configs` order; '0b' = R-14 variant).  The result is
    cached per process (cfg 4 takes 15 s to generate); callers treat it as read-only."""
    key = str(cfg)
    if key not in _MADE:
        _MADE[key] = _make(cfg)
    return _MADE[key]


def _make(cfg: int | str) -> Workload:
    if cfg == "0b":
        idx, variant_b = 0, True
    else:
        idx, variant_b = int(cfg), False
    rng = np.random.Generator(np.random.PCG64(SEED_BASE + idx + (100 if variant_b else 0)))
    if idx == 0:
        atoms = np.array([[0.0, 0.0, 0.0], [1.43, 1.11, 0.0], [-1.43, 1.11, 0.0]])
        kinds = ["O", "H", "H"]
        templates = {"O": [0, 0, 0, 1, 1], "H": [0, 0]}
        if variant_b:
            return _finish("cfg0b", rng, atoms, kinds, templates, 0.1, 1e3, 5, "cfg0", 0.0, nprim_fixed=3)
        e = np.exp(rng.uniform(np.log(0.1), np.log(1e3), size=3))
        c = rng.uniform(0.1, 1.0, size=3)
        return _finish("cfg0", rng, atoms, kinds, templates, 0.1, 1e3, 5, "cfg0", 0.0, shared=(e, c))
    if idx == 1:
        atoms = np.zeros((10, 3))
        atoms[:, 0] = 2.8 * np.arange(10)
        atoms += rng.normal(0.0, 0.1, size=(10, 3))
        kinds = ["H" if i % 2 == 0 else "L" for i in range(10)]
        return _finish("cfg1", rng, atoms, kinds, {"H": HEAVY_SPD, "L": LIGHT_SP}, 0.05, 5e3, 20, "over_nocc", 1e-12)
    if idx in (2, 3):
        atoms, kinds = _lattice60(SEED_BASE + 1000)
        templates = {"H": HEAVY_SPD, "L": LIGHT_SP} if idx == 2 else {"H": HEAVY_SPDF, "L": LIGHT_SPD}
        return _finish(f"cfg{idx}", rng, atoms, kinds, templates, 0.05, 5e3, 120, "over_nocc", 1e-12)
    if idx == 4:
        atoms = _sphere300(rng)
        heavy = set(rng.permutation(300)[:100].tolist())
        kinds = ["H" if i in heavy else "L" for i in range(300)]
        return _finish("cfg4", rng, atoms, kinds, {"H": HEAVY_SPD, "L": LIGHT_SP}, 0.05, 5e3, 600, "trace", 1e-11)
    raise ValueError(f"unknown config {cfg!r}")


def make_custom(atoms, shell_specs, seed, tau=0.0, nocc=None, emin=0.1, emax=50.0, nprim=None):
    """Small ad-hoc systems for class sweeps: shell_specs = [(atom_index, l), ...]; nprim random 1..6
    unless fixed; exponents log-uniform [emin, emax]; D = C C^T / nocc."""
    rng = np.random.Generator(np.random.PCG64(seed))
    atoms = np.ascontiguousarray(atoms, dtype=np.float64)
    s_atom, s_l, s_np, s_off, exps, cofs = [], [], [], [], [], []
    off = 0
    for (ia, l) in shell_specs:
        n = nprim if nprim is not None else int(rng.integers(1, 7))
        e = np.exp(rng.uniform(np.log(emin), np.log(emax), size=n))
        c = rng.uniform(0.1, 1.0, size=n)
        s_atom.append(ia); s_l.append(l); s_np.append(n); s_off.append(off)
        exps.extend(e.tolist()); cofs.extend(c.tolist()); off += n
    nbf = int(sum(ncart(int(l)) for l in s_l))
    nocc = nocc or max(1, nbf // 3)
    D = _density(rng, nbf, nocc, "over_nocc")
    return Workload("custom", atoms, np.array(s_atom, np.int32), np.array(s_l, np.int32),
                    np.array(s_np, np.int32), np.array(s_off, np.int32),
                    np.array(exps, np.float64), np.array(cofs, np.float64), D, tau)


def sparse_density(w, seed, decades=8.0):
    """Input generator of the block-density tests: the workload's D with every shell block scaled by its
    own factor 10^-U(0, decades) (symmetric), so that the block maxima |D|_XY spread over `decades` orders of magnitude
    the way a density difference between two SCF iterations does.  No method arithmetic."""
    rng = np.random.default_rng(seed)
    o = w.bf_offsets()
    f = 10.0 ** (-decades * rng.random((w.nshells, w.nshells)))
    f = np.minimum(f, f.T)
    D = np.array(w.D)
    for X in range(w.nshells):
        for Y in range(w.nshells):
            D[o[X]:o[X + 1], o[Y]:o[Y + 1]] *= f[X, Y]
    return np.ascontiguousarray((D + D.T) / 2)


def perturbed_density(w, seed, atoms=(0,), scale=1e-3):
    """Input generator of the incremental-build tests: D plus a symmetric perturbation of relative size `scale` confined
    to the rows and columns of the basis functions on the given atoms (what one SCF step changes near a site)."""
    rng = np.random.default_rng(seed)
    o = w.bf_offsets()
    on = np.zeros(w.nbf, bool)
    for s in range(w.nshells):
        if int(w.shell_atom[s]) in atoms:
            on[o[s]:o[s + 1]] = True
    P = rng.normal(size=(w.nbf, w.nbf)) * scale * np.abs(w.D).max()
    P = (P + P.T) / 2
    P[~(on[:, None] | on[None, :])] = 0.0
    return np.ascontiguousarray(np.array(w.D) + P)
