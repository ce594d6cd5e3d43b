#!/usr/bin/env python3
"""Code generator for the per-(l_mu,l_nu)-class derivative-integral device functions.

Emits `generated/ris_classes.cuh`: for every class (la >= lb, la <= 3) straight-line CUDA for

  ris_vrr_<la><lb>    one primitive triplet: Obara-Saika vertical recurrence on the bra with the
                      s-type auxiliary function folded in (no ket recurrence),
                        [e+1_i]^(m) = PA_i [e]^(m) + WP_i [e]^(m+1)
                                      + e_i/(2p) ( [e-1_i]^(m) - (rho/p) [e-1_i]^(m+1) ),
                        WP = -(rho/p)(P-C),  [0]^(m) = kappa F_m(T),
                      for e <= E = la+lb+1, followed by the exponent-scaled accumulation of the
                      [e0|s]^(0) classes into the contracted targets
                        acc2a[e] += 2a [e],  e = la+1 .. E      (-> (a+1_i, b|)
                        acc2b[e] += 2b [e],  e = la   .. E      (-> (a, b+1_i|)
                        acc1 [e] +=    [e],  e = max(la-1,0) .. E-2   (-> (a-1_i,b|, (a,b-1_i|)
  ris_hrrc_<la><lb>   one contracted triplet: horizontal recurrence
                        (a, b+1_i| = (a+1_i, b| + (A-B)_i (a, b|
                      on the contracted targets, then
                        d/dA_i (ab|P) = (a+1_i,b|_{2a} - a_i (a-1_i,b|_1
                        d/dB_i (ab|P) = (a,b+1_i|_{2b} - b_i (a,b-1_i|_1
                      contracted on the fly with the D / Gamma^P tile of each state and added to the
                      caller's per-lane accumulator slots (shared memory in the class kernel).

What is computed is Eq. 27 terms 1-2 of the paper for the integrals of Eq. 21
(PAPER.md:119); the evaluation scheme is ours (the paper is silent).  The aux-centre
derivative is NOT generated: the kernels use translational invariance, dC = -(dA + dB).

Numerical stability: the HRR expands (x-B)^k in powers of (x-A); for a primitive pair whose product
centre P sits next to B (b >> a) that expansion cancels by a factor (1 + b/a) per transferred unit.
Every function is therefore generated for BOTH host centres -- "host" (h) carries the VRR, "other" (o)
receives angular momentum through the HRR -- i.e. for all 16 ordered pairs (lh, lo), and the kernels
run the primitive pairs with a >= b hosted on A and those with b > a hosted on B (cancellation <= 2).
In the generated code "a" always means the host: a2 = 2 x host exponent, PA = P - host centre,
AB = host centre - other centre, ga = d/d(host centre), gb = d/d(other centre).  TR selects the tile
element order: false -> (c_host*n_other + c_other), true -> (c_other*n_host + c_host).

Classes whose OTHER shell is an s function (lo = 0, host l = lh > = 0; the kernels run (l,0) pairs with the l shell as
host for EVERY primitive pair) need no transfer at all: the integral is [a 0|, and the derivative with respect to the s
centre is taken by one DIRECT Obara-Saika step on that centre instead of the HRR,
    d/dB_i (a 0|P) = 2b [a, 1_i|,   [a,1_i|^(0) = PB_i [a]^(0) + WP_i [a]^(1) + a_i/(2p) ([a-1_i]^(0) - (rho/p) [a-1_i]^(1)),
with PB = (a/p)(A - B) formed from the exponents (no cancellation for any exponent ratio).  One host phase per pair instead
of two halves the per-pair work (HRR, tile contraction, slot updates) of the (s,s), (p,s), (d,s), (f,s) classes; targets:
    acc2a[e] += 2a [e], e = lh+1;   accbd[a][i] += 2b [a,1_i|, a in comps(lh), i = x,y,z;   acc1[e] += [e], e = lh-1.

Component order inside a shell of degree l: lx descending, then ly descending.
"""
from __future__ import annotations

import os
import sys

LMAX = 3


def comps(l):
    return [(lx, ly, l - lx - ly) for lx in range(l, -1, -1) for ly in range(l - lx, -1, -1)]


_CIDX = {}
for _l in range(0, 2 * LMAX + 3):
    for _k, _c in enumerate(comps(_l)):
        _CIDX[_c] = _k


def cidx(c):
    return _CIDX[tuple(c)]


def nc(l):
    return (l + 1) * (l + 2) // 2


def lower(c, i, k=1):
    c = list(c)
    c[i] -= k
    return tuple(c)


def raise_(c, i):
    c = list(c)
    c[i] += 1
    return tuple(c)


class ClassPlan:
    """Static description of one class: accumulator layout shared by VRR and HRR."""

    def __init__(self, la, lb):
        self.la, self.lb = la, lb
        self.E = la + lb + 1
        self.direct_b = (lb == 0)          # d/dB by a direct OS step on the s centre (see the module docstring)
        self.r2a = list(range(la + 1, self.E + 1))
        self.r2b = [] if self.direct_b else list(range(la, self.E + 1))
        lo = la - 1 if la >= 1 else la
        self.r1 = list(range(lo, self.E - 1)) if (la >= 1 or lb >= 1) else []
        self.off = {}
        n = 0
        for tag, rng in (("2a", self.r2a), ("2b", self.r2b), ("1", self.r1)):
            for e in rng:
                self.off[(tag, e)] = n
                n += nc(e)
        if self.direct_b:
            self.off_bd = n                # accbd[(component of la) * 3 + i]
            n += 3 * nc(la)
        self.nacc = n
        self.fams = [("2a", self.r2a, "a2"), ("2b", self.r2b, "b2"), ("1", self.r1, None)]
        self.vrr_name = f"ris_vrr_{la}{lb}"

    def acc_bd(self, a, i):
        return f"acc[{self.off_bd + 3 * cidx(a) + i}]"

    def acc(self, tag, e, c):
        return f"acc[{self.off[(tag, e)] + cidx(c)}]"


class ClassPlan0:
    """Undifferentiated integrals (mu nu|P) of one class (the fitting step): the VRR stops at
    e = la + lb and the contracted targets are the unscaled [e0|s], e = la .. la+lb."""

    def __init__(self, la, lb):
        self.la, self.lb = la, lb
        self.E = la + lb
        self.r0 = list(range(la, self.E + 1))
        self.off = {}
        n = 0
        for e in self.r0:
            self.off[("0", e)] = n
            n += nc(e)
        self.nacc = n
        self.fams = [("0", self.r0, None)]
        self.vrr_name = f"ris_vrr0_{la}{lb}"

    def acc(self, tag, e, c):
        return f"acc[{self.off[(tag, e)] + cidx(c)}]"


# --------------------------------------------------------------------------- VRR

def gen_vrr(pl: ClassPlan) -> str:
    la, lb, E = pl.la, pl.lb, pl.E
    out = []
    w = out.append
    w(f"// class ({la},{lb}): E={E}, {pl.nacc} contracted targets")
    w("// ACC: the contracted targets -- a double[NACC] array (registers) or any type with operator[] (the class kernel parks")
    w("// part of them in shared memory for the heavy classes)")
    w("template <class ACC>")
    direct = getattr(pl, "direct_b", False)
    w(f"RIS_DEV void {pl.vrr_name}(const double (&F)[{E + 1}], double PA0, double PA1, double PA2,")
    w("    double WP0, double WP1, double WP2, double oo2p, double q, double a2, double b2,")
    w("    ACC& acc" + (", double PB0, double PB1, double PB2)" if direct else ")"))
    w("{")
    PA = ["PA0", "PA1", "PA2"]
    WP = ["WP0", "WP1", "WP2"]
    emin_target = min(rng[0] for _, rng, _ in pl.fams if rng)
    # needed set by backward closure
    need = set()

    def want(e, c, m):
        if (e, c, m) in need:
            return
        need.add((e, c, m))
        if e == 0:
            return
        i = pick_dir(c)
        c1 = lower(c, i)
        want(e - 1, c1, m)
        want(e - 1, c1, m + 1)
        if c[i] >= 2:
            c2 = lower(c, i, 2)
            want(e - 2, c2, m)
            want(e - 2, c2, m + 1)

    def pick_dir(c):
        ones = [i for i in range(3) if c[i] == 1]
        if ones:
            return ones[0]
        nz = [i for i in range(3) if c[i] > 0]
        return min(nz, key=lambda i: c[i])

    for e in range(emin_target, E + 1):
        for c in comps(e):
            want(e, c, 0)
    if direct:                      # [a,1_i|^(0) needs [a]^(0), [a]^(1) and the brackets of [a-1_i]
        for c in comps(la):
            want(la, c, 0)
            want(la, c, 1)
            for i in range(3):
                if c[i] >= 1:
                    want(la - 1, lower(c, i), 0)
                    want(la - 1, lower(c, i), 1)

    def v(e, c, m):
        return "F[%d]" % m if e == 0 else f"v{e}_{cidx(c)}_{m}"

    brackets = set()
    kk = {c[i] - 1 for (e, c, m) in need if e >= 2 for i in [pick_dir(c)] if c[i] >= 2}
    if direct:
        kk |= {c[i] for c in comps(la) for i in range(3) if c[i] >= 1}
    kk = sorted(kk)
    for k in kk:
        w(f"    const double k{k} = {float(k)} * oo2p;")
    for e in range(1, E + 1):
        for m in range(E - e, -1, -1):
            for c in comps(e):
                if (e, c, m) not in need:
                    continue
                i = pick_dir(c)
                c1 = lower(c, i)
                expr = f"fma({PA[i]}, {v(e - 1, c1, m)}, {WP[i]} * {v(e - 1, c1, m + 1)})"
                if c[i] >= 2:
                    c2 = lower(c, i, 2)
                    bn = f"b{e - 2}_{cidx(c2)}_{m}"
                    if bn not in brackets:
                        brackets.add(bn)
                        w(f"    const double {bn} = fma(-q, {v(e - 2, c2, m + 1)}, {v(e - 2, c2, m)});")
                    expr = f"fma(k{c[i] - 1}, {bn}, {expr})"
                w(f"    const double {v(e, c, m)} = {expr};")
        # accumulate level e as soon as it is complete
    for e in range(0, E + 1):
        for c in comps(e):
            val = v(e, c, 0)
            for tag, rng, scale in pl.fams:
                if e not in rng:
                    continue
                if scale:
                    w(f"    {pl.acc(tag, e, c)} = fma({scale}, {val}, {pl.acc(tag, e, c)});")
                else:
                    w(f"    {pl.acc(tag, e, c)} += {val};")
    if direct:
        PB = ["PB0", "PB1", "PB2"]
        for c in comps(la):
            for i in range(3):
                expr = f"fma({PB[i]}, {v(la, c, 0)}, {WP[i]} * {v(la, c, 1)})"
                if c[i] >= 1:
                    c1 = lower(c, i)
                    bn = f"b{la - 1}_{cidx(c1)}_0"
                    if bn not in brackets:
                        brackets.add(bn)
                        w(f"    const double {bn} = fma(-q, {v(la - 1, c1, 1)}, {v(la - 1, c1, 0)});")
                    expr = f"fma(k{c[i]}, {bn}, {expr})"
                w(f"    {pl.acc_bd(c, i)} = fma(b2, {expr}, {pl.acc_bd(c, i)});")
    w("}")
    return "\n".join(out)


# --------------------------------------------------------------------------- HRR + contraction

def gen_hrr_chain(w, pl, tag, la_t, lb_t, prefix, done):
    """Emit (la_t, lb_t| built from acc[tag][e], e = la_t .. la_t+lb_t.  Returns name(ca, cb) for the
    target block; `done` caches emitted intermediates (prefix, e, k, ia, ib)."""

    def name(e, k, a, b):
        if k == 0:
            return pl.acc(tag, e, a)
        return f"{prefix}{e}{k}_{cidx(a)}_{cidx(b)}"

    def build(e, k):
        if k == 0 or (prefix, e, k) in done:
            return
        build(e + 1, k - 1)
        build(e, k - 1)
        done.add((prefix, e, k))
        for a in comps(e):
            for b in comps(k):
                i = max(range(3), key=lambda d: b[d])       # any direction with b_i > 0
                b1 = lower(b, i)
                a1 = raise_(a, i)
                w(f"    const double {name(e, k, a, b)} = fma(AB{i}, {name(e, k - 1, a, b1)}, {name(e + 1, k - 1, a1, b1)});")

    build(la_t, lb_t)
    return lambda a, b: name(la_t, lb_t, a, b)


def gen_hrrc(pl: ClassPlan) -> str:
    la, lb = pl.la, pl.lb
    out = []
    w = out.append
    w(f"// contracted triplet of class ({la},{lb}): HRR, derivative assembly, contraction with the tile of each state,")
    w("// accumulated into the caller's per-lane slots: slot[(s*6 + c)*SL] += sc[s*SC] * g, c = 0..2 centre A, 3..5 centre B")
    w("// (the host centre is B in the TR instantiations).  The tile comes from a provider: ring.get(s) returns the tile of")
    w("// state s (shared-memory ring of the class kernel, or plain memory), element (c_host,c_other) at t[el * ring.es()],")
    w("// el by TR (see gen_classes.py).")
    w("template <bool TR, int SL, int SC, class Ring, class ACC>")
    w(f"RIS_DEV void ris_hrrc_{la}{lb}(const ACC& acc, double AB0, double AB1, double AB2,")
    w("    Ring& ring, int nb, const double* __restrict__ sc, double* __restrict__ slot)")
    w("{")
    done = set()
    X2a = gen_hrr_chain(w, pl, "2a", la + 1, lb, "xa", done)
    Y2b = None if pl.direct_b else gen_hrr_chain(w, pl, "2b", la, lb + 1, "yb", done)
    X1m = gen_hrr_chain(w, pl, "1", la - 1, lb, "xm", done) if la >= 1 else None
    Y1m = gen_hrr_chain(w, pl, "1", la, lb - 1, "xm", done) if lb >= 1 else None
    nca, ncb = nc(la), nc(lb)
    w("    constexpr int OH = TR ? 3 : 0, OO = TR ? 0 : 3;")
    w("    const size_t estride = ring.es();")
    w("    for (int s = 0; s < nb; ++s) {")
    w("        const double* __restrict__ t = ring.get(s);")
    w("        double ga0 = 0.0, ga1 = 0.0, ga2 = 0.0, gb0 = 0.0, gb1 = 0.0, gb2 = 0.0;")
    for ia, a in enumerate(comps(la)):
        for ib, b in enumerate(comps(lb)):
            w(f"        {{ const double w = t[(TR ? {ib * nca + ia} : {ia * ncb + ib}) * estride];")
            for i in range(3):
                w(f"          ga{i} = fma(w, {X2a(raise_(a, i), b)}, ga{i});")
                if a[i] >= 1:
                    w(f"          ga{i} = fma(-{float(a[i])} * w, {X1m(lower(a, i), b)}, ga{i});")
                gbv = pl.acc_bd(a, i) if pl.direct_b else Y2b(a, raise_(b, i))
                w(f"          gb{i} = fma(w, {gbv}, gb{i});")
                if b[i] >= 1:
                    w(f"          gb{i} = fma(-{float(b[i])} * w, {Y1m(a, lower(b, i))}, gb{i});")
            w("        }")
    w("        const double c = SC ? sc[s * SC] : 1.0;       // SC = 0: no scale (K type)")
    w("        double* __restrict__ o = slot + s * 6 * SL;")
    for i in range(3):
        w(f"        o[(OH + {i}) * SL] = fma(c, ga{i}, o[(OH + {i}) * SL]);")
    for i in range(3):
        w(f"        o[(OO + {i}) * SL] = fma(c, gb{i}, o[(OO + {i}) * SL]);")
    w("    }")
    w("}")
    return "\n".join(out)


def gen_hrr0c(pl: ClassPlan0) -> str:
    la, lb = pl.la, pl.lb
    out = []
    w = out.append
    w(f"// contracted undifferentiated triplet of class ({la},{lb}): HRR to (a b|P), dot with the tile of each state:")
    w("// slot[s*SL] += sum_{ab} tile_s[el] (ab|P).  Tile element order as in ris_hrrc (TR).")
    w("template <bool TR, int SL>")
    w(f"RIS_DEV void ris_hrr0c_{la}{lb}(const double (&acc)[{pl.nacc}], double AB0, double AB1, double AB2,")
    w("    const double* __restrict__ tile, size_t estride, size_t sstride, int nb, double* __restrict__ slot)")
    w("{")
    done = set()
    X = gen_hrr_chain(w, pl, "0", la, lb, "x", done)
    nca, ncb = nc(la), nc(lb)
    w("    for (int s = 0; s < nb; ++s) {")
    w("        const double* __restrict__ t = tile + (size_t)s * sstride;")
    w("        double v = 0.0;")
    for ia, a in enumerate(comps(la)):
        for ib, b in enumerate(comps(lb)):
            w(f"        v = fma(t[(TR ? {ib * nca + ia} : {ia * ncb + ib}) * estride], {X(a, b)}, v);")
    w("        slot[s * SL] += v;")
    w("    }")
    w("}")
    return "\n".join(out)


def gen_hrr0w(pl: ClassPlan0) -> str:
    la, lb = pl.la, pl.lb
    out = []
    w = out.append
    w(f"// contracted undifferentiated triplet of class ({la},{lb}): HRR to (a b|P), ADDED to out[el * estride] (the two")
    w("// host-centre phases of a pair add into the same, pre-zeroed elements).  Element order by TR as in ris_hrrc.")
    w("template <bool TR>")
    w(f"RIS_DEV void ris_hrr0w_{la}{lb}(const double (&acc)[{pl.nacc}], double AB0, double AB1, double AB2,")
    w("    double* __restrict__ out, size_t estride)")
    w("{")
    done = set()
    X = gen_hrr_chain(w, pl, "0", la, lb, "x", done)
    nca, ncb = nc(la), nc(lb)
    for ia, a in enumerate(comps(la)):
        for ib, b in enumerate(comps(lb)):
            w(f"    out[(TR ? {ib * nca + ia} : {ia * ncb + ib}) * estride] += {X(a, b)};")
    w("}")
    return "\n".join(out)



# --------------------------------------------------------------------------- p-type auxiliary functions (NEXT-2)
# PAPER.md:125 ("a single GTO for each angular momentum component (up to l = 2) on each atom"), PAPER.md:168 ("s- and
# p-type for Coulomb").  The aux function is (r-C)_i exp(-alpha |r-C|^2); one more Obara-Saika step, on the aux centre,
#   [a b|p_i]^(m) = WC_i [a b|s]^(m+1) + a_i/(2(p+alpha)) [a-1_i b|s]^(m+1) + b_i/(2(p+alpha)) [a b-1_i|s]^(m+1),
#   WC = W - C = (1 - rho/p)(P - C),
# turns the s-aux integrals of one Boys order higher into the targets; the bra HRR and the contraction code are the ones
# of the s-aux class (same target layout).  Emission is a memoised recursion over ([a], b in {0, 1_j}, ket in {s, p_i}, m).

class Emitter:
    def __init__(self, w, direct_names):
        self.w = w
        self.memo = {}
        self.dn = direct_names     # argument names: PA, WP, PB lists, WC scalar name, ...

    def k(self, n):                # n / (2p)
        return f"k{n}"

    def get(self, a, b, ket, m):
        """name of [a b|ket]^(m); a: bra triple on the host; b: None or direction j of a p function on the other (s) centre;
        ket: None (s aux) or direction i (p aux)."""
        key = (a, b, ket, m)
        if key in self.memo:
            return self.memo[key]
        w = self.w
        if ket is not None:
            i = ket
            terms = [f"WC * {self.get(a, b, None, m + 1)}"]
            if a[i] >= 1:
                terms.append(f"{float(a[i])} * oo2pa * {self.get(lower(a, i), b, None, m + 1)}")
            if b == i:
                terms.append(f"oo2pa * {self.get(a, None, None, m + 1)}")
            name = f"t{sum(a)}_{cidx(a)}_{'n' if b is None else b}_{m}"
            w(f"    const double {name} = " + " + ".join(terms) + ";")
        elif b is not None:
            j = b
            expr = f"fma(PB{j}, {self.get(a, None, None, m)}, WP{j} * {self.get(a, None, None, m + 1)})"
            if a[j] >= 1:
                expr = f"fma({self.k(a[j])}, {self.bracket(lower(a, j), m)}, {expr})"
            name = f"u{sum(a)}_{cidx(a)}_{j}_{m}"
            w(f"    const double {name} = {expr};")
        elif sum(a) == 0:
            name = f"F[{m}]"
        else:
            ones = [d for d in range(3) if a[d] == 1]
            d = ones[0] if ones else min((x for x in range(3) if a[x] > 0), key=lambda x: a[x])
            a1 = lower(a, d)
            expr = f"fma(PA{d}, {self.get(a1, None, None, m)}, WP{d} * {self.get(a1, None, None, m + 1)})"
            if a[d] >= 2:
                expr = f"fma({self.k(a[d] - 1)}, {self.bracket(lower(a, d, 2), m)}, {expr})"
            name = f"v{sum(a)}_{cidx(a)}_{m}"
            w(f"    const double {name} = {expr};")
        self.memo[key] = name
        return name

    def bracket(self, a, m):
        key = ("br", a, m)
        if key not in self.memo:
            name = f"b{sum(a)}_{cidx(a)}_{m}"
            self.w(f"    const double {name} = fma(-q, {self.get(a, None, None, m + 1)}, {self.get(a, None, None, m)});")
            self.memo[key] = name
        return self.memo[key]


def gen_vrr_p(pl, i: int) -> str:
    """VRR + accumulation of the targets [e0|p_i] (and, for the direct classes, 2b [a,1_j|p_i]) of plan `pl` (ClassPlan or
    ClassPlan0) for the p aux component i.  F holds kappa F_m, m = 0 .. E+1."""
    la, lb, E = pl.la, pl.lb, pl.E
    direct = getattr(pl, "direct_b", False)
    out = []
    w = out.append
    w(f"// class ({la},{lb}), p-type aux component {i}: {pl.nacc} contracted targets")
    w("template <class ACC>")
    w(f"RIS_DEV void {pl.vrr_name.replace('ris_vrr', 'ris_vrrp')}_{i}(const double (&F)[{E + 2}], double PA0, double PA1, double PA2,")
    w("    double WP0, double WP1, double WP2, double oo2p, double q, double a2, double b2,")
    w("    ACC& acc, double WC, double oo2pa" + (", double PB0, double PB1, double PB2)" if direct else ")"))
    w("{")
    for n in range(1, E + 2):
        w(f"    const double k{n} = {float(n)} * oo2p;")
    em = Emitter(w, None)
    for e in range(0, E + 1):
        for c in comps(e):
            val = None
            for tag, rng, scale in pl.fams:
                if e not in rng:
                    continue
                if val is None:
                    val = em.get(c, None, i, 0)
                if scale:
                    w(f"    {pl.acc(tag, e, c)} = fma({scale}, {val}, {pl.acc(tag, e, c)});")
                else:
                    w(f"    {pl.acc(tag, e, c)} += {val};")
    if direct:
        for c in comps(la):
            for j in range(3):
                w(f"    {pl.acc_bd(c, j)} = fma(b2, {em.get(c, j, i, 0)}, {pl.acc_bd(c, j)});")
    w("}")
    return "\n".join(out)


def generate() -> str:
    parts = ["// GENERATED by gen_classes.py -- do not edit.  See that file for the recurrences.",
             "#pragma once", ""]
    classes = [(la, lb) for la in range(LMAX + 1) for lb in range(LMAX + 1)]
    for la, lb in classes:
        pl = ClassPlan(la, lb)
        parts.append(f"template <> struct RisClass<{la},{lb}> {{ static constexpr int E = {pl.E}; "
                     f"static constexpr int NACC = {pl.nacc}; static constexpr int NCA = {nc(la)}; "
                     f"static constexpr int NCB = {nc(lb)}; }};")
        p0 = ClassPlan0(la, lb)
        parts.append(f"template <> struct RisClass0<{la},{lb}> {{ static constexpr int E = {p0.E}; "
                     f"static constexpr int NACC = {p0.nacc}; }};")
    parts.append("")
    for la, lb in classes:
        pl = ClassPlan(la, lb)
        parts.append(gen_vrr(pl))
        parts.append("")
        parts.append(gen_hrrc(pl))
        parts.append("")
        p0 = ClassPlan0(la, lb)
        parts.append(gen_vrr(p0))
        parts.append("")
        parts.append(gen_hrr0c(p0))
        parts.append("")
        parts.append(gen_hrr0w(p0))
        parts.append("")
        for i in range(3):
            parts.append(gen_vrr_p(pl, i))
            parts.append("")
            parts.append(gen_vrr_p(p0, i))
            parts.append("")
    # dispatch helpers
    parts.append("template <int LA, int LB, class... A> RIS_DEV void ris_vrr(A&&... a) {")
    for la, lb in classes:
        parts.append(f"    if constexpr (LA == {la} && LB == {lb}) ris_vrr_{la}{lb}(static_cast<A&&>(a)...);")
    parts.append("}")
    parts.append("template <int LA, int LB, class... A> RIS_DEV void ris_vrr0(A&&... a) {")
    for la, lb in classes:
        parts.append(f"    if constexpr (LA == {la} && LB == {lb}) ris_vrr0_{la}{lb}(static_cast<A&&>(a)...);")
    parts.append("}")
    for nm in ("ris_vrrp", "ris_vrrp0"):
        parts.append(f"template <int LA, int LB, int DIR, class... A> RIS_DEV void {nm}(A&&... a) {{")
        for la, lb in classes:
            for i in range(3):
                parts.append(f"    if constexpr (LA == {la} && LB == {lb} && DIR == {i}) {nm}_{la}{lb}_{i}(static_cast<A&&>(a)...);")
        parts.append("}")
    parts.append("template <int LA, int LB, bool TR, int SL, class... A> RIS_DEV void ris_hrr0c(A&&... a) {")
    for la, lb in classes:
        parts.append(f"    if constexpr (LA == {la} && LB == {lb}) ris_hrr0c_{la}{lb}<TR, SL>(static_cast<A&&>(a)...);")
    parts.append("}")
    parts.append("template <int LA, int LB, bool TR, class... A> RIS_DEV void ris_hrr0w(A&&... a) {")
    for la, lb in classes:
        parts.append(f"    if constexpr (LA == {la} && LB == {lb}) ris_hrr0w_{la}{lb}<TR>(static_cast<A&&>(a)...);")
    parts.append("}")
    parts.append("template <int LA, int LB, bool TR, int SL, int SC, class... A> RIS_DEV void ris_hrrc(A&&... a) {")
    for la, lb in classes:
        parts.append(f"    if constexpr (LA == {la} && LB == {lb}) ris_hrrc_{la}{lb}<TR, SL, SC>(static_cast<A&&>(a)...);")
    parts.append("}")
    return "\n".join(parts) + "\n"


def main():
    here = os.path.dirname(os.path.abspath(__file__))
    outdir = os.path.join(here, "generated")
    os.makedirs(outdir, exist_ok=True)
    path = os.path.join(outdir, "ris_classes.cuh")
    text = generate()
    if not os.path.exists(path) or open(path).read() != text:
        with open(path, "w") as f:
            f.write(text)
    return path


if __name__ == "__main__":
    print(main())
