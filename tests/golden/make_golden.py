"""Writes the stored expected values of the big configs.  Calls ONLY oracle/ and the seeded input generator
(paper_2406_11185_b200/workloads.py, which holds no method arithmetic); never the CUDA path.

    python tests/golden/make_golden.py full 2            # full oracle J, K, Q, counts, energies of cfg 2
    python tests/golden/make_golden.py full 3            # same for cfg 3 (hours; resumable: --ckpt, --max-seconds)
    python tests/golden/make_golden.py full 3 --ckpt a.npz --chunk-lo 0 --chunk-hi 100     # part of the chunks on one machine,
    python tests/golden/make_golden.py full 3 --ckpt b.npz --chunk-lo 100 --chunk-hi 256   # the rest on another,
    python tests/golden/make_golden.py merge 3 a.npz b.npz                                 # then add the partial sums
    python tests/golden/make_golden.py blocks 4 [--per-type 23]   # stratified sampled J/K shell blocks of cfg 4

`full` runs oracle.jk_range (orc_jk's own loop, restricted to a range of bra pairs, long double partial sums) chunk
by chunk, checkpoints the running long double sums after every chunk, and finally rounds once to fp64: the result is
what oracle.jk returns.  Stored (npz): the lower triangles of J and K, the Schwarz table Q, Dmax, kept / unique /
primitive-quartet counts, per-class counts, E_J = 1/2 tr(DJ) and E_K = -1/4 tr(DK) (long double sums), and the
SHA-256 of the input arrays (tests refuse a golden file whose hash differs from the workload they regenerate).

`blocks` evaluates J and K shell blocks (A, B) one by one from the definition with the same screen
(oracle.jk_block), stratified so that every ordered block type (l_A, l_B) appears `--per-type` times
("~200 random shell pairs"); element parity on samples, energy parity NOT claimed (cfg 4's full
oracle is a day of CPU time).
"""
from __future__ import annotations

import argparse
import hashlib
import os
import sys
import time

import numpy as np

HERE = os.path.dirname(os.path.abspath(__file__))
ROOT = os.path.dirname(os.path.dirname(HERE))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

import oracle                                             # noqa: E402
from paper_2406_11185_b200 import workloads as W          # noqa: E402


def input_sha256(w) -> str:
    """Hash of everything both sides read: geometry, shells, raw exponents/coefficients, D, tau."""
    h = hashlib.sha256()
    for a in (w.atoms, w.shell_atom, w.shell_l, w.shell_nprim, w.shell_off, w.exponents, w.coefficients, w.D,
              np.array([w.tau])):
        a = np.ascontiguousarray(a)
        h.update(str(a.dtype).encode()); h.update(str(a.shape).encode()); h.update(a.tobytes())
    return h.hexdigest()


def chunk_bounds(npair: int, nchunks: int):
    """Bra-pair ranges of roughly equal work (a bra pair pab has pab+1 candidate ket pairs)."""
    edges = [int(round(npair * np.sqrt(k / nchunks))) for k in range(nchunks + 1)]
    edges[0], edges[-1] = 0, npair
    return [(edges[k], edges[k + 1]) for k in range(nchunks) if edges[k + 1] > edges[k]]


def save_partial(path, sha, nchunks, lo, done, cnt, cc, J, K):
    """Running long double sums of the chunks [lo, done): long double does not survive np.save portably, so the file
    keeps hi + lo fp64 parts (106 bits, more than the 64-bit significand of the x87 type)."""
    Jhi = J.astype(np.float64); Khi = K.astype(np.float64)
    tmp = path + ".tmp.npz"
    np.savez(tmp, sha=sha, nchunks=nchunks, lo=lo, done=done, cnt=cnt, cc=cc, Jhi=Jhi,
             Jlo=(J - Jhi).astype(np.float64), Khi=Khi, Klo=(K - Khi).astype(np.float64))
    os.replace(tmp, path)


def write_full(out, cfg, w, sha, Q, J, K, cnt, cc, seconds):
    """Round the long double sums once and store the result (what oracle.jk returns)."""
    N = J.shape[0]
    Dl = np.asarray(w.D, np.longdouble)
    EJ = 0.5 * np.sum(Dl * J); EK = -0.25 * np.sum(Dl * K)
    J64 = J.astype(np.float64); K64 = K.astype(np.float64)
    assert np.array_equal(J64, J64.T) or np.abs(J64 - J64.T).max() <= 1e-13 * np.abs(J64).max()
    il = np.tril_indices(N)
    np.savez_compressed(out, sha=sha, cfg=cfg, nbf=N, tau=w.tau, dmax=oracle.dmax(w.D), Q=Q,
                        J_tril=J64[il], K_tril=K64[il], unique=cnt[0], kept=cnt[1], prim=cnt[2], per_class=cc,
                        EJ_hi=np.float64(EJ), EJ_lo=np.float64(EJ - np.longdouble(np.float64(EJ))),
                        EK_hi=np.float64(EK), EK_lo=np.float64(EK - np.longdouble(np.float64(EK))),
                        seconds=seconds, threads=oracle.num_threads())
    print(f"wrote {out}: kept {cnt[1]} prim {cnt[2]} E_J {float(EJ):.12f} E_K {float(EK):.12f} {seconds:.0f} s", flush=True)


def merge(cfg: int, out: str, parts):
    """Add the partial sums of `full --chunk-lo/--chunk-hi` runs (each a finished --ckpt file) and write the result."""
    w = W.make(cfg)
    sha = input_sha256(w)
    bs = oracle.basis_from_workload(w)
    N = bs.nbf
    J = np.zeros((N, N), np.longdouble); K = np.zeros((N, N), np.longdouble)
    cnt = np.zeros(3, np.int64); cc = np.zeros(oracle.NQCLASS, np.int64)
    ranges = []
    nch = None
    for path in parts:
        c = np.load(path, allow_pickle=False)
        assert str(c["sha"]) == sha, f"{path} was made from other inputs"
        nch = int(c["nchunks"]) if nch is None else nch
        assert int(c["nchunks"]) == nch, "partial files use different chunkings"
        ranges.append((int(c["lo"]), int(c["done"])))
        J += c["Jhi"].astype(np.longdouble) + c["Jlo"].astype(np.longdouble)
        K += c["Khi"].astype(np.longdouble) + c["Klo"].astype(np.longdouble)
        cnt += c["cnt"]; cc[:len(c["cc"])] += c["cc"]        # files written before the g classes existed hold 55 entries
    ranges.sort()
    assert ranges[0][0] == 0 and ranges[-1][1] == nch and all(a[1] == b[0] for a, b in zip(ranges, ranges[1:])), \
        f"partial files do not tile the chunks 0..{nch}: {ranges}"
    write_full(out, cfg, w, sha, oracle.schwarz(bs), J, K, cnt, cc, 0.0)


def full(cfg: int, out: str, ckpt: str, nchunks: int, max_seconds: float = 0.0, chunk_lo: int = 0, chunk_hi: int = -1):
    w = W.make(cfg)
    sha = input_sha256(w)
    bs = oracle.basis_from_workload(w)
    t0 = time.time()
    Q = oracle.schwarz(bs)
    print(f"cfg {cfg}: N={bs.nbf} shells={bs.nshells} threads={oracle.num_threads()} schwarz {time.time() - t0:.1f} s", flush=True)
    npair = bs.nshells * (bs.nshells + 1) // 2
    chunks = chunk_bounds(npair, nchunks)
    N = bs.nbf
    J = np.zeros((N, N), np.longdouble); K = np.zeros((N, N), np.longdouble)
    cnt = np.zeros(3, np.int64); cc = np.zeros(oracle.NQCLASS, np.int64)
    chunk_hi = len(chunks) if chunk_hi < 0 else min(chunk_hi, len(chunks))
    done = chunk_lo
    if ckpt and os.path.exists(ckpt):
        c = np.load(ckpt, allow_pickle=False)
        if str(c["sha"]) == sha and int(c["nchunks"]) == len(chunks) and int(c["lo"]) == chunk_lo:
            J = c["Jhi"].astype(np.longdouble) + c["Jlo"].astype(np.longdouble)
            K = c["Khi"].astype(np.longdouble) + c["Klo"].astype(np.longdouble)
            cnt, done = c["cnt"], int(c["done"])
            cc[:len(c["cc"])] = c["cc"]
            print(f"resuming after chunk {done}/{len(chunks)}", flush=True)
    for i in range(done, chunk_hi):
        if max_seconds and time.time() - t0 > max_seconds:
            print(f"stopping after {time.time() - t0:.0f} s with {i}/{len(chunks)} chunks done (resume with the same --ckpt)", flush=True)
            return
        lo, hi = chunks[i]
        t1 = time.time()
        j, k, ci = oracle.jk_range(bs, w.D, w.tau, Q, lo, hi)
        J += j; K += k
        cnt += np.array([ci["unique"], ci["kept"], ci["prim"]], np.int64); cc += ci["per_class"]
        print(f"chunk {i + 1}/{len(chunks)} pab [{lo},{hi}) kept {ci['kept']} prim {ci['prim']} "
              f"{time.time() - t1:.0f} s (total {time.time() - t0:.0f} s)", flush=True)
        if ckpt:
            save_partial(ckpt, sha, len(chunks), chunk_lo, i + 1, cnt, cc, J, K)
    if chunk_lo != 0 or chunk_hi != len(chunks):
        print(f"chunks [{chunk_lo},{chunk_hi}) done; combine the partial files with `merge`", flush=True)
        return
    write_full(out, cfg, w, sha, Q, J, K, cnt, cc, time.time() - t0)


def blocks(cfg: int, out: str, per_type: int, seed: int):
    w = W.make(cfg)
    sha = input_sha256(w)
    bs = oracle.basis_from_workload(w)
    t0 = time.time()
    Q = oracle.schwarz(bs)
    dm = oracle.dmax(w.D)
    cnt = oracle.count(bs, Q, dm, w.tau)
    rng = np.random.default_rng(seed)
    ls = sorted(set(int(x) for x in bs.l))
    by_l = {l: np.flatnonzero(bs.l == l) for l in ls}
    picks = []
    for la in ls:
        for lb in ls:
            seen = set()
            while len(seen) < per_type:
                seen.add((int(rng.choice(by_l[la])), int(rng.choice(by_l[lb]))))
            picks += sorted(seen)
    nmax = max(bs.ncart)
    AB = np.array(picks, np.int32)
    Jb = np.zeros((len(picks), nmax, nmax)); Kb = np.zeros((len(picks), nmax, nmax))
    for i, (A, B) in enumerate(picks):
        j, k = oracle.jk_block(bs, w.D, w.tau, Q, dm, A, B)
        Jb[i, :j.shape[0], :j.shape[1]] = j; Kb[i, :k.shape[0], :k.shape[1]] = k
        if (i + 1) % 20 == 0:
            print(f"block {i + 1}/{len(picks)} {time.time() - t0:.0f} s", flush=True)
    np.savez_compressed(out, sha=sha, cfg=cfg, nbf=bs.nbf, tau=w.tau, dmax=dm, Q=Q, AB=AB, J_blocks=Jb, K_blocks=Kb,
                        unique=cnt["unique"], kept=cnt["kept"], prim=cnt["prim"], per_class=cnt["per_class"],
                        seconds=time.time() - t0, threads=oracle.num_threads())
    print(f"wrote {out}: {len(picks)} blocks, {time.time() - t0:.0f} s", flush=True)


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("mode", choices=["full", "blocks", "merge"])
    ap.add_argument("cfg", type=int)
    ap.add_argument("parts", nargs="*", help="`merge`: the finished --ckpt files of the partial runs")
    ap.add_argument("--chunk-lo", type=int, default=0, help="`full`: first chunk of a partial run")
    ap.add_argument("--chunk-hi", type=int, default=-1, help="`full`: one past the last chunk of a partial run")
    ap.add_argument("--out", default=None)
    ap.add_argument("--ckpt", default=None, help="checkpoint file of a `full` run (resumed if it matches the inputs)")
    ap.add_argument("--chunks", type=int, default=64)
    ap.add_argument("--max-seconds", type=float, default=0.0, help="`full`: stop (checkpointed) before a chunk once this much time has passed")
    ap.add_argument("--per-type", type=int, default=23)
    ap.add_argument("--seed", type=int, default=2406)
    a = ap.parse_args()
    if a.mode == "full":
        full(a.cfg, a.out or os.path.join(HERE, f"cfg{a.cfg}_full.npz"), a.ckpt, a.chunks, a.max_seconds, a.chunk_lo, a.chunk_hi)
    elif a.mode == "merge":
        merge(a.cfg, a.out or os.path.join(HERE, f"cfg{a.cfg}_full.npz"), a.parts)
    else:
        blocks(a.cfg, a.out or os.path.join(HERE, f"cfg{a.cfg}_blocks.npz"), a.per_type, a.seed)


if __name__ == "__main__":
    main()
