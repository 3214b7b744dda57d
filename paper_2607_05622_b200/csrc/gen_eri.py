#!/usr/bin/env python3
"""Code generator for the Obara-Saika / Head-Gordon-Pople shell-quartet recurrences (step a7).

Emits `eri_gen.h`: straight-line fp64 code, one VRR routine per canonical quartet class
(la>=lb, lc>=ld, braclass>=ketclass; l <= 2 -> 21 classes) and one HRR routine per pair class (6).
The paper's integral engine is generated the same way ("HGP-OS ... VRR-A -> VRR-C -> HRR-AB -> HRR-CD",
PAPER.md:L318, L336 Fig. 6; fully unrolled regime for s/p/d, L316).  Nothing here is taken from the
CPU oracle, which uses McMurchie-Davidson Hermite recurrences instead.

Recurrences (textbook Obara-Saika, primitive quartet, [e0|f0]^(m) with e on centre A, f on centre C):
  [e+1_i,0|00]^(m) = PA_i [e0|00]^(m) + WP_i [e0|00]^(m+1)
                     + e_i/(2p) ( [e-1_i,0|00]^(m) - (rho/p) [e-1_i,0|00]^(m+1) )
  [e0|f+1_i,0]^(m) = QC_i [e0|f0]^(m) + WQ_i [e0|f0]^(m+1)
                     + f_i/(2q) ( [e0|f-1_i,0]^(m) - (rho/q) [e0|f-1_i,0]^(m+1) )
                     + e_i/(2(p+q)) [e-1_i,0|f0]^(m+1)
  [00|00]^(m)      = K_ab K_cd 2 pi^{5/2} / (p q sqrt(p+q)) F_m(rho |PQ|^2)        (supplied as F[m])
HRR on contracted integrals:
  (a, b+1_i| = (a+1_i, b| + (A_i - B_i) (a, b|        and the same on the ket with C - D.

Usage: python gen_eri.py <out_dir>
"""
from __future__ import annotations

import sys
from pathlib import Path

LMAX = 2
AX = "xyz"


def comps(l):
    return [(i, j, l - i - j) for i in range(l, -1, -1) for j in range(l - i, -1, -1)]


def ncart(l):
    return (l + 1) * (l + 2) // 2


def range_index(lo, hi):
    """index of Cartesian components of degrees lo..hi concatenated"""
    idx = {}
    for deg in range(lo, hi + 1):
        for c in comps(deg):
            idx[c] = len(idx)
    return idx


def dec(v, i):
    w = list(v)
    w[i] -= 1
    return tuple(w)


def inc(v, i):
    w = list(v)
    w[i] += 1
    return tuple(w)


def mulc(n, name):
    return name if n == 1 else "(%d.0*%s)" % (n, name)


class VRR:
    def __init__(self, la, lb, lc, ld):
        self.la, self.lb, self.lc, self.ld = la, lb, lc, ld
        self.memo = {}
        self.dmemo = {}
        self.lines = []
        self.n = 0

    def new(self, expr):
        name = "v%d" % self.n
        self.n += 1
        self.lines.append("const double %s = %s;" % (name, expr))
        return name

    def node(self, e, f, m):
        if min(e) < 0 or min(f) < 0:
            return None
        if sum(e) == 0 and sum(f) == 0:
            return "F[%d]" % m
        key = (e, f, m)
        if key in self.memo:
            return self.memo[key]
        if sum(f) > 0:
            # choose the axis with the fewest terms
            best = None
            for i in range(3):
                if f[i] == 0:
                    continue
                cost = 2 + (2 if f[i] > 1 else 0) + (1 if e[i] > 0 else 0)
                if best is None or cost < best[0]:
                    best = (cost, i)
            i = best[1]
            f1 = dec(f, i)
            a0 = self.node(e, f1, m)
            a1 = self.node(e, f1, m + 1)
            expr = "QC%s*%s + WQ%s*%s" % (AX[i], a0, AX[i], a1)
            if f1[i] > 0:
                d = self.diff(e, dec(f1, i), m, "rq")
                expr += " + %s*%s" % (mulc(f1[i], "oo2q"), d)
            if e[i] > 0:
                c = self.node(dec(e, i), f1, m + 1)
                expr += " + %s*%s" % (mulc(e[i], "oo2pq"), c)
        else:
            best = None
            for i in range(3):
                if e[i] == 0:
                    continue
                cost = 2 + (2 if e[i] > 1 else 0)
                if best is None or cost < best[0]:
                    best = (cost, i)
            i = best[1]
            e1 = dec(e, i)
            a0 = self.node(e1, f, m)
            a1 = self.node(e1, f, m + 1)
            expr = "PA%s*%s + WP%s*%s" % (AX[i], a0, AX[i], a1)
            if e1[i] > 0:
                d = self.diff(dec(e1, i), f, m, "rp")
                expr += " + %s*%s" % (mulc(e1[i], "oo2p"), d)
        name = self.new(expr)
        self.memo[key] = name
        return name

    def diff(self, e, f, m, r):
        key = (e, f, m, r)
        if key in self.dmemo:
            return self.dmemo[key]
        a0 = self.node(e, f, m)
        a1 = self.node(e, f, m + 1)
        name = self.new("%s - %s*%s" % (a0, r, a1))
        self.dmemo[key] = name
        return name

    def generate(self):
        la, lb, lc, ld = self.la, self.lb, self.lc, self.ld
        eidx = range_index(la, la + lb)
        fidx = range_index(lc, lc + ld)
        nf = len(fidx)
        # every target is accumulated right after it is computed (short live ranges: fewer registers held)
        for e, ie in eidx.items():
            for f, jf in fidx.items():
                v = self.node(e, f, 0)
                self.lines.append("sink.template put<%d>(%s);" % (ie * nf + jf, v))
        return self.lines, len(eidx), nf


def gen_hrr(la, lb):
    """(a b| for |a|=la, |b|=lb from (e 0|, la<=|e|<=la+lb.  src[eidx*ss], dst[(ia*nb+ib)*ds]."""
    eidx = range_index(la, la + lb)
    memo = {}
    lines = []
    cnt = [0]

    def H(a, b):
        if sum(b) == 0:
            return "src[%d*ss]" % eidx[a]
        key = (a, b)
        if key in memo:
            return memo[key]
        i = [k for k in range(3) if b[k] > 0][0]
        b1 = dec(b, i)
        x = H(inc(a, i), b1)
        y = H(a, b1)
        name = "h%d" % cnt[0]
        cnt[0] += 1
        lines.append("const double %s = %s + AB%s*%s;" % (name, x, AX[i], y))
        memo[key] = name
        return name

    outs = []
    ca, cb = comps(la), comps(lb)
    for ia, a in enumerate(ca):
        for ib, b in enumerate(cb):
            outs.append("dst[%d*ds] = %s;" % (ia * len(cb) + ib, H(a, b)))
    return lines + outs


PAIR_CLASSES = [(0, 0), (1, 0), (1, 1), (2, 0), (2, 1), (2, 2)]


def main(out_dir):
    out = Path(out_dir)
    out.mkdir(parents=True, exist_ok=True)
    hdr = []
    hdr.append("// GENERATED by gen_eri.py -- do not edit.  Obara-Saika VRR / HGP HRR straight-line code (see gen_eri.py).")
    hdr.append("#pragma once")
    hdr.append("namespace ltjk_gen {")
    hdr.append("template<int LA,int LB> struct Hrr;")
    for (la, lb) in PAIR_CLASSES:
        body = gen_hrr(la, lb)
        hdr.append("template<> struct Hrr<%d,%d> {" % (la, lb))
        hdr.append("  static constexpr int NE = %d;  // components of degrees la..la+lb" % len(range_index(la, la + lb)))
        hdr.append("  static constexpr int NAB = %d;" % (ncart(la) * ncart(lb)))
        hdr.append("  LTJK_HD static void run(const double* __restrict__ src, const int ss, double* __restrict__ dst, "
                   "const int ds, const double ABx, const double ABy, const double ABz) {")
        hdr.append("    (void)ABx; (void)ABy; (void)ABz;")
        for ln in body:
            hdr.append("    " + ln)
        hdr.append("  }")
        hdr.append("};")
    hdr.append("struct AccSink { double* __restrict__ acc; template<int I> LTJK_HD void put(const double v) { acc[I] += v; } };")
    hdr.append("template<int LA,int LB,int LC,int LD> struct Vrr;")
    stats = []
    for ib_, (la, lb) in enumerate(PAIR_CLASSES):
        for ik_, (lc, ld) in enumerate(PAIR_CLASSES):
            if ik_ > ib_:
                continue
            g = VRR(la, lb, lc, ld)
            body, ne, nf = g.generate()
            stats.append(((la, lb, lc, ld), g.n, ne * nf))
            hdr.append("template<> struct Vrr<%d,%d,%d,%d> {" % (la, lb, lc, ld))
            hdr.append("  static constexpr int NE = %d, NF = %d, NNODE = %d;" % (ne, nf, g.n))
            # the targets are handed, in increasing index order, to a sink: `AccSink` adds them to a per-thread array
            # (one thread per quartet), the cooperative kernels reduce them across the lanes of a half-warp instead
            hdr.append("  template<class SINK> LTJK_HD static void run_t(const double* __restrict__ F, "
                       "const double PAx, const double PAy, const double PAz, "
                       "const double WPx, const double WPy, const double WPz, "
                       "const double QCx, const double QCy, const double QCz, "
                       "const double WQx, const double WQy, const double WQz, "
                       "const double oo2p, const double oo2q, const double oo2pq, "
                       "const double rp, const double rq, SINK& sink) {")
            hdr.append("    (void)PAx;(void)PAy;(void)PAz;(void)WPx;(void)WPy;(void)WPz;(void)QCx;(void)QCy;(void)QCz;"
                       "(void)WQx;(void)WQy;(void)WQz;(void)oo2p;(void)oo2q;(void)oo2pq;(void)rp;(void)rq;")
            for ln in body:
                hdr.append("    " + ln)
            hdr.append("  }")
            hdr.append("  LTJK_HD static void run(const double* __restrict__ F, "
                       "const double PAx, const double PAy, const double PAz, "
                       "const double WPx, const double WPy, const double WPz, "
                       "const double QCx, const double QCy, const double QCz, "
                       "const double WQx, const double WQy, const double WQz, "
                       "const double oo2p, const double oo2q, const double oo2pq, "
                       "const double rp, const double rq, double* __restrict__ acc) {")
            hdr.append("    AccSink s{acc};")
            hdr.append("    run_t(F, PAx, PAy, PAz, WPx, WPy, WPz, QCx, QCy, QCz, WQx, WQy, WQz, oo2p, oo2q, oo2pq, rp, rq, s);")
            hdr.append("  }")
            hdr.append("};")
    hdr.append("} // namespace ltjk_gen")
    (out / "eri_gen.h").write_text("\n".join(hdr) + "\n")
    # ---- classes with ONE index raised to l = 3, for the first-derivative builds (ltjk_grad.cu):
    # d/dA_x of a shell of l is a shell of l + 1 (and one of l - 1), so (f b|c d) with b, c, d <= 2 is all that is needed.
    d1 = ["// GENERATED by gen_eri.py -- do not edit.  f-raised classes for the derivative builds (see gen_eri.py).",
          "#pragma once", "namespace ltjk_gen {"]
    for lb in range(LMAX + 1):
        body = gen_hrr(LMAX + 1, lb)
        d1.append("template<> struct Hrr<%d,%d> {" % (LMAX + 1, lb))
        d1.append("  static constexpr int NE = %d;" % len(range_index(LMAX + 1, LMAX + 1 + lb)))
        d1.append("  static constexpr int NAB = %d;" % (ncart(LMAX + 1) * ncart(lb)))
        d1.append("  LTJK_HD static void run(const double* __restrict__ src, const int ss, double* __restrict__ dst, "
                  "const int ds, const double ABx, const double ABy, const double ABz) {")
        d1.append("    (void)ABx; (void)ABy; (void)ABz;")
        for ln in body:
            d1.append("    " + ln)
        d1.append("  }")
        d1.append("};")
    for lb in range(LMAX + 1):
        for (lc, ld) in PAIR_CLASSES:
            g = VRR(LMAX + 1, lb, lc, ld)
            body, ne, nf = g.generate()
            stats.append(((LMAX + 1, lb, lc, ld), g.n, ne * nf))
            d1.append("template<> struct Vrr<%d,%d,%d,%d> {" % (LMAX + 1, lb, lc, ld))
            d1.append("  static constexpr int NE = %d, NF = %d, NNODE = %d;" % (ne, nf, g.n))
            d1.append("  template<class SINK> LTJK_HD static void run_t(const double* __restrict__ F, "
                      "const double PAx, const double PAy, const double PAz, "
                      "const double WPx, const double WPy, const double WPz, "
                      "const double QCx, const double QCy, const double QCz, "
                      "const double WQx, const double WQy, const double WQz, "
                      "const double oo2p, const double oo2q, const double oo2pq, "
                      "const double rp, const double rq, SINK& sink) {")
            d1.append("    (void)PAx;(void)PAy;(void)PAz;(void)WPx;(void)WPy;(void)WPz;(void)QCx;(void)QCy;(void)QCz;"
                      "(void)WQx;(void)WQy;(void)WQz;(void)oo2p;(void)oo2q;(void)oo2pq;(void)rp;(void)rq;")
            for ln in body:
                d1.append("    " + ln)
            d1.append("  }")
            d1.append("  LTJK_HD static void run(const double* __restrict__ F, "
                      "const double PAx, const double PAy, const double PAz, "
                      "const double WPx, const double WPy, const double WPz, "
                      "const double QCx, const double QCy, const double QCz, "
                      "const double WQx, const double WQy, const double WQz, "
                      "const double oo2p, const double oo2q, const double oo2pq, "
                      "const double rp, const double rq, double* __restrict__ acc) {")
            d1.append("    AccSink s{acc};")
            d1.append("    run_t(F, PAx, PAy, PAz, WPx, WPy, WPz, QCx, QCy, QCz, WQx, WQy, WQz, oo2p, oo2q, oo2pq, rp, rq, s);")
            d1.append("  }")
            d1.append("};")
    d1.append("} // namespace ltjk_gen")
    (out / "eri_gen_d1.h").write_text("\n".join(d1) + "\n")
    with open(out / "eri_gen_stats.txt", "w") as fh:
        fh.write("# class(la lb lc ld)  vrr_nodes_per_primitive_quartet  contracted_accumulators\n")
        for cls, n, na in stats:
            fh.write("%d%d%d%d %d %d\n" % (cls + (n, na)))
    return 0


if __name__ == "__main__":
    sys.exit(main(sys.argv[1] if len(sys.argv) > 1 else str(Path(__file__).resolve().parent / "gen")))
