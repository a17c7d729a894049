#!/usr/bin/env python3
"""Code generator for the per-class ERI device code (product code; run by the build).

"For each type of angular momentum combination, we optimize and determine a unique computational path
through code generation".  This script is that step for sm_100a: for a quartet class
(la lb|lc ld), la>=lb, lc>=ld, it walks the Obara-Saika recurrences (Head-Gordon-Pople form; the paper
names HGP, and prints no equations, so the textbook recurrences are restated in
DESIGN.md) top-down from the needed targets [e0|f0]^(0), e in la..la+lb, f in lc..lc+ld, keeps only the
intermediates that are reached, and emits

  * G_<abcd>::vrr()      straight-line fp64 code for one primitive quartet, accumulating the contraction
                         into acc[NE*NF] (registers when the class is small enough, else local memory);
  * G_<abcd>::hrr()      the horizontal recurrences on the contracted [e0|f0] and one `put` per integral
                         (the digestion functor of the caller folds it into J and K);
  * exact FP64 instruction counts of those paths (the "model flops" of the roofline).

The same DAG can be evaluated in Python (`VrrDag.evaluate`, `HrrDag.evaluate`), which is how
tests/test_codegen.py checks the generator on CPU before anything runs on a GPU.
"""
from __future__ import annotations

import argparse
import json
import os
from collections import OrderedDict

AX = "xyz"


def comps(l):
    return [(x, y, l - x - y) for x in range(l, -1, -1) for y in range(l - x, -1, -1)]


def ncart(l):
    return (l + 1) * (l + 2) // 2


def dec(t, i):
    u = list(t); u[i] -= 1
    return tuple(u)


def inc(t, i):
    u = list(t); u[i] += 1
    return tuple(u)


ZERO = (0, 0, 0)


def choose_dir(vec, how):
    nz = [i for i in range(3) if vec[i] > 0]
    if how == "first":
        return nz[0]
    if how == "last":
        return nz[-1]
    if how == "max":
        return max(nz, key=lambda i: (vec[i], -i))
    if how == "min":
        return min(nz, key=lambda i: (vec[i], i))
    raise ValueError(how)


def all_targets(la, lb, lc, ld):
    """(a, c) of every contracted [e0|f0] the HRR needs, in global accumulator order."""
    return [(a, c) for dega in range(la, la + lb + 1) for a in comps(dega)
            for degc in range(lc, lc + ld + 1) for c in comps(degc)]


class VrrDag:
    """Vertical recurrences for one primitive quartet.

    bra:  [a+1_i,0|00]^(m) = PA_i [a|0]^(m) + WP_i [a|0]^(m+1) + a_i/(2 zeta) ( [a-1_i|0]^(m) - rho/zeta [a-1_i|0]^(m+1) )
    ket:  [a0|c+1_i,0]^(m) = QC_i [a|c]^(m) + WQ_i [a|c]^(m+1) + c_i/(2 eta) ( [a|c-1_i]^(m) - rho/eta [a|c-1_i]^(m+1) )
                             + a_i/(2(zeta+eta)) [a-1_i|c]^(m+1)
    """

    def __init__(self, la, lb, lc, ld, how="first", targets=None):
        self.la, self.lb, self.lc, self.ld = la, lb, lc, ld
        self.lab, self.lcd = la + lb, lc + ld
        self.L = self.lab + self.lcd
        self.how = how
        self.nodes = OrderedDict()       # key -> spec ; insertion order is a valid topological order
        if targets is None:              # all [e0|f0], in acc order
            targets = all_targets(la, lb, lc, ld)
        self.targets = list(targets)     # (a, c); position in this list = accumulator index of the pass
        for (a, c) in self.targets:
            self._need(("V", a, c, 0))
        self.ids = {k: i for i, k in enumerate(self.nodes)}

    def _need(self, key):
        if key in self.nodes:
            return
        kind = key[0]
        if kind == "T":                  # T = V(m) - r * V(m+1)
            _, a, c, m, side = key
            self._need(("V", a, c, m)); self._need(("V", a, c, m + 1))
            self.nodes[key] = ("T", side, ("V", a, c, m), ("V", a, c, m + 1))
            return
        _, a, c, m = key
        if a == ZERO and c == ZERO:
            self.nodes[key] = ("B", m)
            return
        if c != ZERO:
            i = choose_dir(c, self.how)
            cm = dec(c, i)
            d0, d1 = ("V", a, cm, m), ("V", a, cm, m + 1)
            self._need(d0); self._need(d1)
            t2 = None; tx = None
            if cm[i] > 0:
                t2 = ("T", a, dec(cm, i), m, "ket"); self._need(t2)
            if a[i] > 0:
                tx = ("V", dec(a, i), cm, m + 1); self._need(tx)
            self.nodes[key] = ("K", i, d0, d1, cm[i], t2, a[i], tx)
        else:
            i = choose_dir(a, self.how)
            am = dec(a, i)
            d0, d1 = ("V", am, c, m), ("V", am, c, m + 1)
            self._need(d0); self._need(d1)
            t2 = None
            if am[i] > 0:
                t2 = ("T", dec(am, i), c, m, "bra"); self._need(t2)
            self.nodes[key] = ("A", i, d0, d1, am[i], t2)

    def fused_targets(self):
        """Targets no other node reads: their recurrence is accumulated straight into the contracted sum,
        acc = fma(PA, d0, acc); acc = fma(WP, d1, acc); ..., one instruction fewer than value + add."""
        used = set()
        for s in self.nodes.values():
            if s[0] == "T":
                used.update((s[2], s[3]))
            elif s[0] == "A":
                used.update(k for k in (s[2], s[3], s[5]) if k)
            elif s[0] == "K":
                used.update(k for k in (s[2], s[3], s[5], s[7]) if k)
        return {("V", a, c, 0) for (a, c) in self.targets
                if ("V", a, c, 0) not in used and self.nodes[("V", a, c, 0)][0] in ("A", "K")}

    # ---- FP64 operation count per primitive quartet of the recurrence in its canonical form (every node a value, one
    # add per contracted target; DMUL/DFMA/DADD each count 1): the MODEL count of DESIGN.md R-21, unchanged since round 1.
    # The emitted code executes len(fused_targets()) instructions fewer (fp64_instr).
    def fp64_instr(self):
        return self.fp64_ops() - len(self.fused_targets())

    def fp64_ops(self):
        n = 0
        for spec in self.nodes.values():
            if spec[0] == "B":
                n += 1                      # scale F_m by the prefactor
            elif spec[0] == "T":
                n += 1
            elif spec[0] == "A":
                n += 2 + (1 if spec[5] else 0)
            elif spec[0] == "K":
                n += 2 + (1 if spec[5] else 0) + (1 if spec[7] else 0)
        return n + len(self.targets)        # + contraction adds

    def max_m(self):
        return max(s[1] for s in self.nodes.values() if s[0] == "B")

    # ---- reference evaluation of the DAG in Python (float or mpmath numbers) ----
    def evaluate(self, ctx):
        """ctx: dict with PA, WP, QC, WQ (3-vectors), inv2z, inv2e, inv2ze, roz, roe, F (list, already scaled)."""
        val = {}
        for key, s in self.nodes.items():
            if s[0] == "B":
                val[key] = ctx["F"][s[1]]
            elif s[0] == "T":
                r = ctx["roz"] if s[1] == "bra" else ctx["roe"]
                val[key] = val[s[2]] - r * val[s[3]]
            elif s[0] == "A":
                _, i, d0, d1, n2, t2 = s
                v = ctx["PA"][i] * val[d0] + ctx["WP"][i] * val[d1]
                if t2:
                    v += n2 * ctx["inv2z"] * val[t2]
                val[key] = v
            else:
                _, i, d0, d1, n2, t2, nx, tx = s
                v = ctx["QC"][i] * val[d0] + ctx["WQ"][i] * val[d1]
                if t2:
                    v += n2 * ctx["inv2e"] * val[t2]
                if tx:
                    v += nx * ctx["inv2ze"] * val[tx]
                val[key] = v
        return [val[("V", a, c, 0)] for (a, c) in self.targets]

    # ---- CUDA emission ----
    def emit(self, out):
        name = lambda k: f"v{self.ids[k]}"
        used_z, used_e, used_ze = set(), set(), set()
        for s in self.nodes.values():
            if s[0] == "A" and s[5]:
                used_z.add(s[4])
            if s[0] == "K":
                if s[5]:
                    used_e.add(s[4])
                if s[7]:
                    used_ze.add(s[6])
        for n in sorted(used_z):
            out.append(f"    const R kz{n} = R({float(n)}) * c.inv2z;")
        for n in sorted(used_e):
            out.append(f"    const R ke{n} = R({float(n)}) * c.inv2e;")
        for n in sorted(used_ze):
            out.append(f"    const R kx{n} = R({float(n)}) * c.inv2ze;")
        tgt_index = {("V", a, cc, 0): j for j, (a, cc) in enumerate(self.targets)}
        fused = self.fused_targets()
        for key, s in self.nodes.items():
            v = name(key)
            if key in fused:
                t = tgt_index[key]
                if s[0] == "A":
                    _, i, d0, d1, n2, t2 = s
                    terms = [(f"c.PA{AX[i]}", name(d0)), (f"c.WP{AX[i]}", name(d1))] + ([(f"kz{n2}", name(t2))] if t2 else [])
                else:
                    _, i, d0, d1, n2, t2, nx, tx = s
                    terms = [(f"c.QC{AX[i]}", name(d0)), (f"c.WQ{AX[i]}", name(d1))] + ([(f"ke{n2}", name(t2))] if t2 else []) \
                        + ([(f"kx{nx}", name(tx))] if tx else [])
                for (x, y) in terms:
                    out.append(f"    acc.template fma<{t}>({x}, {y});")
                continue
            if s[0] == "B":
                out.append(f"    const R {v} = F[{s[1]}];")
            elif s[0] == "T":
                r = "c.roz" if s[1] == "bra" else "c.roe"
                out.append(f"    const R {v} = fma(-{r}, {name(s[3])}, {name(s[2])});")
            elif s[0] == "A":
                _, i, d0, d1, n2, t2 = s
                e = f"fma(c.PA{AX[i]}, {name(d0)}, c.WP{AX[i]} * {name(d1)})"
                if t2:
                    e = f"fma(kz{n2}, {name(t2)}, {e})"
                out.append(f"    const R {v} = {e};")
            else:
                _, i, d0, d1, n2, t2, nx, tx = s
                e = f"fma(c.QC{AX[i]}, {name(d0)}, c.WQ{AX[i]} * {name(d1)})"
                if t2:
                    e = f"fma(ke{n2}, {name(t2)}, {e})"
                if tx:
                    e = f"fma(kx{nx}, {name(tx)}, {e})"
                out.append(f"    const R {v} = {e};")
            if key in tgt_index:
                out.append(f"    acc.template add<{tgt_index[key]}>({v});")


class HrrDag:
    """Horizontal recurrences on contracted integrals:
         (a, b+1_i| c) = (a+1_i, b| c) + (A_i-B_i)(a b| c);   (ab| c, d+1_i) = (ab| c+1_i, d) + (C_i-D_i)(ab| c d)."""

    def __init__(self, la, lb, lc, ld, diag_only=False, how="first"):
        self.la, self.lb, self.lc, self.ld = la, lb, lc, ld
        self.how = how
        self.tindex = {}
        j = 0
        for dega in range(la, la + lb + 1):
            for a in comps(dega):
                for degc in range(lc, lc + ld + 1):
                    for c in comps(degc):
                        self.tindex[(a, c)] = j; j += 1
        self.nodes = OrderedDict()
        self.outputs = []     # (ia, ib, ic, id, key)
        A, B, C, D = comps(la), comps(lb), comps(lc), comps(ld)
        for ia, a in enumerate(A):
            for ib, b in enumerate(B):
                for ic, c in enumerate(C):
                    for idd, d in enumerate(D):
                        if diag_only and not (ia == ic and ib == idd):
                            continue
                        key = ("H2", a, b, c, d)
                        self._need(key)
                        self.outputs.append((ia, ib, ic, idd, key))
        self.ids = {k: i for i, k in enumerate(self.nodes)}

    def _need(self, key):
        if key in self.nodes:
            return
        if key[0] == "H2":
            _, a, b, c, d = key
            if d == ZERO:
                k1 = ("H1", a, b, c); self._need(k1)
                self.nodes[key] = ("alias", k1)
                return
            i = choose_dir(d, self.how)
            dm = dec(d, i)
            k0, k1 = ("H2", a, b, inc(c, i), dm), ("H2", a, b, c, dm)
            self._need(k0); self._need(k1)
            self.nodes[key] = ("hrr", "CD", i, k0, k1)
        else:
            _, a, b, c = key
            if b == ZERO:
                self.nodes[key] = ("acc", self.tindex[(a, c)])
                return
            i = choose_dir(b, self.how)
            bm = dec(b, i)
            k0, k1 = ("H1", inc(a, i), bm, c), ("H1", a, bm, c)
            self._need(k0); self._need(k1)
            self.nodes[key] = ("hrr", "AB", i, k0, k1)

    def fp64_ops(self):
        return sum(1 for s in self.nodes.values() if s[0] == "hrr")

    def evaluate(self, acc, AB, CD):
        val = {}
        for key, s in self.nodes.items():
            if s[0] == "acc":
                val[key] = acc[s[1]]
            elif s[0] == "alias":
                val[key] = val[s[1]]
            else:
                _, which, i, k0, k1 = s
                g = AB if which == "AB" else CD
                val[key] = val[k0] + g[i] * val[k1]
        return {(ia, ib, ic, idd): val[k] for (ia, ib, ic, idd, k) in self.outputs}

    def emit(self, out):
        def name(k):
            s = self.nodes[k]
            if s[0] == "acc":
                return f"acc.template get<{s[1]}>()"
            if s[0] == "alias":
                return name(s[1])
            return f"h{self.ids[k]}"
        # emit H1 nodes first, then per-(a,b) groups of H2 nodes followed by their puts
        emitted = set()

        def emit_node(k):
            if k in emitted:
                return
            s = self.nodes[k]
            if s[0] == "acc":
                emitted.add(k); return
            if s[0] == "alias":
                emit_node(s[1]); emitted.add(k); return
            _, which, i, k0, k1 = s
            emit_node(k0); emit_node(k1)
            out.append(f"    const R h{self.ids[k]} = fma({which}{AX[i]}, {name(k1)}, {name(k0)});")
            emitted.add(k)

        for (ia, ib, ic, idd, k) in self.outputs:
            emit_node(k)
            out.append(f"    dg.template put<{ia},{ib},{ic},{idd}>({name(k)});")


def class_tag(la, lb, lc, ld):
    return f"{la}{lb}{lc}{ld}"


def best_vrr(la, lb, lc, ld, targets=None):
    best = None
    for how in ("first", "last", "max", "min"):
        d = VrrDag(la, lb, lc, ld, how, targets)
        if best is None or d.fp64_instr() < best.fp64_instr():
            best = d
    return best


PREAMBLE_OPS = 70     # geometry, prefactor and Boys of one primitive quartet, repeated in every pass


def plan_passes(la, lb, lc, ld, cmax):
    """Multi-pass pruned VRR: partition the [e0|f0] targets into chunks of at most ~cmax accumulators (a chunk =
    a group of bra degrees x a run of ket components) and re-walk, per chunk, only the part of the DAG it needs.
    Returns the list of VrrDag (one per pass) with the smallest total FP64 op count among a few partitions."""
    edegs = list(range(la, la + lb + 1))
    clist = [c for degc in range(lc, lc + ld + 1) for c in comps(degc)]
    best, best_cost = None, None
    for egroups in ([edegs], [[d] for d in edegs]):
        passes = []
        for eg in egroups:
            alist = [a for d in eg for a in comps(d)]
            g = max(1, cmax // len(alist))
            for i in range(0, len(clist), g):
                tg = [(a, c) for a in alist for c in clist[i:i + g]]
                passes.append(best_vrr(la, lb, lc, ld, tg))
        cost = sum(p.fp64_instr() + PREAMBLE_OPS for p in passes)
        if best is None or cost < best_cost:
            best, best_cost = passes, cost
    return best


def generate_class(la, lb, lc, ld, cmax_list=()):
    tag = class_tag(la, lb, lc, ld)
    vrr = best_vrr(la, lb, lc, ld)
    hrr = HrrDag(la, lb, lc, ld)
    NE = sum(ncart(e) for e in range(la, la + lb + 1))
    NF = sum(ncart(f) for f in range(lc, lc + ld + 1))
    nint = ncart(la) * ncart(lb) * ncart(lc) * ncart(ld)
    o = []
    o.append(f"// GENERATED by csrc/gen/gen_eri.py -- class ({'spdf'[la]}{'spdf'[lb]}|{'spdf'[lc]}{'spdf'[ld]}); do not edit.")
    o.append(f"// VRR: {len(vrr.nodes)} nodes, {vrr.fp64_ops()} FP64 operations per primitive quartet in canonical form (the model count), "
             f"{vrr.fp64_instr()} instructions emitted (direction rule '{vrr.how}');")
    o.append(f"// HRR: {hrr.fp64_ops()} FP64 ops per contracted quartet; {nint} integrals.")
    o.append("#pragma once")
    o.append(f"struct G_{tag} {{")
    o.append(f"    static constexpr int LA = {la}, LB = {lb}, LC = {lc}, LD = {ld};")
    o.append(f"    static constexpr int NA = {ncart(la)}, NB = {ncart(lb)}, NC = {ncart(lc)}, ND = {ncart(ld)};")
    o.append(f"    static constexpr int NE = {NE}, NF = {NF}, NACC = {NE * NF}, MMAX = {vrr.max_m()};")
    o.append(f"    static constexpr int VRR_OPS = {vrr.fp64_ops()}, HRR_OPS = {hrr.fp64_ops()}, NINT = {nint};")
    o.append("    // R = the arithmetic type (double, or float for the single-precision band of the mixed-precision dispatch)")
    o.append("    template <class Ctx, class Acc, class R>")
    o.append("    static __device__ __forceinline__ void vrr(const Ctx &c, const R *__restrict__ F, Acc &acc) {")
    vrr.emit(o)
    o.append("    }")
    o.append("    template <class Acc, class Dg, class R>")
    o.append("    static __device__ __forceinline__ void hrr(const Acc &acc, R ABx, R ABy, R ABz, R CDx, R CDy, R CDz, Dg &dg) {")
    hrr.emit(o)
    o.append("    }")
    o.append("};")
    gidx = {t: i for i, t in enumerate(all_targets(la, lb, lc, ld))}
    pass_meta = {}
    for cmax in cmax_list:
        passes = plan_passes(la, lb, lc, ld, cmax)
        if len(passes) < 2:
            continue
        tot = sum(p.fp64_ops() for p in passes)
        pass_meta[str(cmax)] = {"npass": len(passes), "vrr_ops": tot, "max_chunk": max(len(p.targets) for p in passes)}
        o.append(f"// multi-pass pruned VRR, chunks of <= {cmax} accumulators: {len(passes)} passes, {tot} FP64 ops per primitive quartet")
        o.append(f"struct GP_{tag}_{cmax} {{")
        o.append(f"    static constexpr int NPASS = {len(passes)};")
        o.append(f"    static constexpr int NCHUNK_MAX = {max(len(p.targets) for p in passes)};")
        o.append("    static __host__ __device__ constexpr int pass_nacc(int P) { constexpr int t[] = {" + ", ".join(str(len(p.targets)) for p in passes) + "}; return t[P]; }")
        o.append("    static __host__ __device__ constexpr int pass_mmax(int P) { constexpr int t[] = {" + ", ".join(str(p.max_m()) for p in passes) + "}; return t[P]; }")
        o.append("    template <int P, class Ctx, class Acc, class R>")
        o.append("    static __device__ __forceinline__ void vrr_pass(const Ctx &c, const R *__restrict__ F, Acc &acc) {")
        for k, pdag in enumerate(passes):
            o.append(f"      if constexpr (P == {k}) {{")
            pdag.emit(o)
            o.append("      }")
        o.append("    }")
        o.append("    template <int P, class Chunk, class Acc>")
        o.append("    static __device__ __forceinline__ void store_pass(const Chunk &ch, Acc &acc) {")
        for k, pdag in enumerate(passes):
            o.append(f"      if constexpr (P == {k}) {{")
            for i, t in enumerate(pdag.targets):
                o.append(f"        acc.template set<{gidx[t]}>(ch.template get<{i}>());")
            o.append("      }")
        o.append("    }")
        o.append("};")
    meta = {"tag": tag, "l": [la, lb, lc, ld], "vrr_ops": vrr.fp64_ops(), "hrr_ops": hrr.fp64_ops(), "nint": nint,
            "nacc": NE * NF, "vrr_nodes": len(vrr.nodes), "how": vrr.how, "passes": pass_meta}
    return "\n".join(o) + "\n", meta


PAIR_CLASSES = [(la, lb) for la in range(5) for lb in range(la + 1)]      # pc = la(la+1)/2+lb, 15 classes (up to g)


def all_classes(lmax=3):
    out = []
    pcs = [p for p in PAIR_CLASSES if p[0] <= lmax]
    for X, (la, lb) in enumerate(pcs):
        for Y, (lc, ld) in enumerate(pcs[:X + 1]):
            out.append((la, lb, lc, ld))
    return out


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--out", required=True)
    ap.add_argument("--max-nacc", type=int, default=1000, help="largest NE*NF emitted as straight-line code")
    ap.add_argument("--max-l2-nacc", type=int, default=1000, help="the same limit for classes without f shells")
    ap.add_argument("--max-l", type=int, default=2, help="highest shell l emitted as straight-line code")
    ap.add_argument("--cmax", type=str, default="{}", help="JSON {tag: [chunk sizes]} of multi-pass variants to emit")
    args = ap.parse_args()
    os.makedirs(args.out, exist_ok=True)
    cmax_map = json.loads(args.cmax)
    metas = []
    for (la, lb, lc, ld) in all_classes(3):
        NE = sum(ncart(e) for e in range(la, la + lb + 1))
        NF = sum(ncart(f) for f in range(lc, lc + ld + 1))
        if max(la, lb, lc, ld) > args.max_l or NE * NF > (args.max_nacc if la == 3 else args.max_l2_nacc):
            continue
        src, meta = generate_class(la, lb, lc, ld, cmax_map.get(class_tag(la, lb, lc, ld), ()))
        with open(os.path.join(args.out, f"eri_{meta['tag']}.cuh"), "w") as f:
            f.write(src)
        metas.append(meta)
    with open(os.path.join(args.out, "classes.json"), "w") as f:
        json.dump(metas, f, indent=1)
    # angular momenta and FP64 instruction counts of ALL classes (also those that run through the Rys kernels):
    # the library's class table and its model-flop count read this list
    with open(os.path.join(args.out, "class_meta.inc"), "w") as f:
        f.write("// GENERATED: ADFT_CLASS_META(qc, la, lb, lc, ld, vrr_ops, hrr_ops, nint)\n")
        for (la, lb, lc, ld) in all_classes(4):
            X, Y = la * (la + 1) // 2 + lb, lc * (lc + 1) // 2 + ld
            # (the g classes only need the counts; one direction rule keeps the generation time down)
            v = best_vrr(la, lb, lc, ld) if la < 4 else VrrDag(la, lb, lc, ld, "first")
            h = HrrDag(la, lb, lc, ld)
            f.write(f"ADFT_CLASS_META({X * (X + 1) // 2 + Y}, {la}, {lb}, {lc}, {ld}, {v.fp64_ops()}, {h.fp64_ops()}, "
                    f"{ncart(la) * ncart(lb) * ncart(lc) * ncart(ld)})\n")
    # X-macro list of straight-line classes
    with open(os.path.join(args.out, "classes.inc"), "w") as f:
        f.write("// GENERATED: ADFT_GEN_CLASS(la, lb, lc, ld, tag)\n")
        for m in metas:
            la, lb, lc, ld = m["l"]
            f.write(f"ADFT_GEN_CLASS({la}, {lb}, {lc}, {ld}, {m['tag']})\n")
    print(f"generated {len(metas)} classes into {args.out}")


if __name__ == "__main__":
    main()
