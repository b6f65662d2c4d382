#!/usr/bin/env python
"""Generates line_codelets.cuh: straight-line fp64 code for the lattice line operators of PAPER.md Eqs. 49-50.

For a periodic line of N real samples with unit spacing the two operators are
    D  = F^-1 (i k) F   with the Nyquist mode zeroed,      D2 = F^-1 (-k^2) F,
k_j = 2 pi j / N (j < N/2), 2 pi (j - N) / N otherwise (Eq. 44).  Both are REAL matrices, so a complex line is two
independent real lines (real and imaginary part) and every transform is a real-input FFT (N/2 + 1 complex bins).
The kernels (fft_plane_kernels.cuh) give one thread one real line in registers and call

    inner(x) -> a = D x, b = D2 x          one real-to-complex FFT, two complex-to-real FFTs sharing the spectrum
    outer(g, q) -> c = D g + D2 q          two real-to-complex FFTs, spectra combined, one complex-to-real FFT

This script writes each of them as a branch-free sequence of DADD / DMUL / DFMA on named temporaries (the compiler
keeps everything in registers): a mixed-radix (2, 3, 4, 5) Cooley-Tukey network is built symbolically on the real
and imaginary parts; every intermediate is identified by the LINEAR FORM it computes, so equal (or opposite) values
are computed once -- which removes the redundant half of a real-input / Hermitian-input transform and the
multiplications by 0, +-1, +-i automatically -- unused values are dropped, multiplications are fused into the
following additions (DFMA), and several factorisation orders are tried, keeping the one with the fewest fp64
instructions.  The result is checked here against the dense operator matrices built from the defining sums.

The physical spacing dx enters as D / dx and D2 / dx^2; the kernels fold those factors into the staged potentials.
Nothing here is shared with oracle/ (which builds dense matrices from the DFT sums and applies them directly).
"""
import itertools
import math
import os
import sys

import numpy as np

TOL = 1e-9
LINE_SIZES = (4, 6, 8, 10, 12, 16, 20, 24, 32, 40)


def cis(num, den):
    """exp(2 pi i num / den) = (cos, sin), with the argument reduced to the first octant so that symmetric twiddles
    are bitwise symmetric."""
    num %= den
    if num == 0:
        return 1.0, 0.0
    if 8 * num <= den:
        th = 2.0 * math.pi * num / den
        return math.cos(th), math.sin(th)
    if 4 * num <= den:                                    # (pi/4, pi/2]: reflect about pi/4
        c, s = cis(den - 4 * num, 4 * den)
        return s, c
    if 2 * num <= den:                                    # (pi/2, pi]: reflect about pi/2
        c, s = cis(den - 2 * num, 2 * den)
        return -c, s
    c, s = cis(den - num, den)                            # lower half plane: conjugate
    return c, -s


class Dag:
    """linear straight-line program over `nin` real inputs; values are signed references (node, sign) or None = 0."""

    def __init__(self, nin):
        self.nin = nin
        self.kind, self.args, self.form = [], [], []
        self.table = {}
        self.inputs = [self._new("in", (i,), np.eye(nin, dtype=np.longdouble)[i]) for i in range(nin)]

    def _key(self, f):
        nz = np.flatnonzero(np.abs(f) > TOL)
        if nz.size == 0:
            return None, 0
        s = 1 if f[nz[0]] > 0 else -1
        return tuple(np.round((f * s).astype(np.float64), 9)), s

    def _new(self, kind, args, form):
        key, s = self._key(form)
        nid = len(self.kind)
        self.kind.append(kind); self.args.append(args); self.form.append(form)
        self.table[key] = (nid, s)
        return (nid, 1)

    def _lookup(self, form):
        key, s = self._key(form)
        if key is None:
            return "zero"
        hit = self.table.get(key)
        if hit is None:
            return None
        nid, s0 = hit
        return (nid, s * s0)

    def valform(self, r):
        return None if r is None else self.form[r[0]] * r[1]

    def add(self, a, b):
        if a is None:
            return b
        if b is None:
            return a
        form = self.valform(a) + self.valform(b)
        hit = self._lookup(form)
        if hit == "zero":
            return None
        if hit is not None:
            return hit
        (na, sa), (nb, sb) = a, b
        if sa == 1 and sb == 1:
            return self._new("add", (na, nb), form)
        if sa == 1 and sb == -1:
            return self._new("sub", (na, nb), form)
        if sa == -1 and sb == 1:
            return self._new("sub", (nb, na), form)
        n, _ = self._new("add", (na, nb), -form)
        return (n, -1)

    def sub(self, a, b):
        return self.add(a, self.neg(b))

    @staticmethod
    def neg(a):
        return None if a is None else (a[0], -a[1])

    def mul(self, c, a):
        if a is None or abs(c) < 1e-15:
            return None
        if abs(c - 1.0) < 1e-15:
            return a
        if abs(c + 1.0) < 1e-15:
            return self.neg(a)
        n, s = a
        if self.kind[n] == "mul":
            c0, n0 = self.args[n]
            return self.mul(c * s * c0, (n0, 1))
        form = self.form[n] * (c * s)
        hit = self._lookup(form)
        if hit == "zero":
            return None
        if hit is not None:
            return hit
        return self._new("mul", (c * s, n), form)


# ---- symbolic complex arithmetic on (re, im) pairs of signed references ----
def c_add(d, x, y):
    return (d.add(x[0], y[0]), d.add(x[1], y[1]))


def c_sub(d, x, y):
    return (d.sub(x[0], y[0]), d.sub(x[1], y[1]))


def c_mulc(d, w, x):
    wr, wi = w
    return (d.sub(d.mul(wr, x[0]), d.mul(wi, x[1])), d.add(d.mul(wr, x[1]), d.mul(wi, x[0])))


def c_muli(d, x, sgn):
    """x * (sgn i)"""
    return (d.mul(-sgn, x[1]), d.mul(sgn, x[0]))


def c_scale(d, c, x):
    return (d.mul(c, x[0]), d.mul(c, x[1]))


def small_dft(d, t, sgn):
    """DFT of len(t) in {2, 3, 4, 5} points with kernel exp(sgn 2 pi i j p / r)."""
    r = len(t)
    if r == 2:
        return [c_add(d, t[0], t[1]), c_sub(d, t[0], t[1])]
    if r == 4:
        a0, a1 = c_add(d, t[0], t[2]), c_sub(d, t[0], t[2])
        b0, b1 = c_add(d, t[1], t[3]), c_muli(d, c_sub(d, t[1], t[3]), sgn)
        return [c_add(d, a0, b0), c_add(d, a1, b1), c_sub(d, a0, b0), c_sub(d, a1, b1)]
    if r == 3:
        s = c_add(d, t[1], t[2])
        df = c_sub(d, t[1], t[2])
        y0 = c_add(d, t[0], s)
        m = c_add(d, t[0], c_scale(d, -0.5, s))
        e = c_muli(d, c_scale(d, math.sqrt(3.0) / 2.0, df), sgn)
        return [y0, c_add(d, m, e), c_sub(d, m, e)]
    if r == 5:
        c1, s1 = cis(1, 5)
        c2, s2 = cis(2, 5)
        a1, a2 = c_add(d, t[1], t[4]), c_add(d, t[2], t[3])
        b1, b2 = c_sub(d, t[1], t[4]), c_sub(d, t[2], t[3])
        y0 = c_add(d, t[0], c_add(d, a1, a2))
        m1 = c_add(d, t[0], c_add(d, c_scale(d, c1, a1), c_scale(d, c2, a2)))
        m2 = c_add(d, t[0], c_add(d, c_scale(d, c2, a1), c_scale(d, c1, a2)))
        e1 = c_muli(d, c_add(d, c_scale(d, s1, b1), c_scale(d, s2, b2)), sgn)
        e2 = c_muli(d, c_sub(d, c_scale(d, s2, b1), c_scale(d, s1, b2)), sgn)
        return [y0, c_add(d, m1, e1), c_add(d, m2, e2), c_sub(d, m2, e2), c_sub(d, m1, e1)]
    raise ValueError(r)


def fft(d, xs, sgn, radices, dif):
    """X[k] = sum_n xs[n] exp(sgn 2 pi i n k / N); radices: the radix used at each recursion level."""
    n = len(xs)
    if n == 1:
        return list(xs)
    r = radices[0]
    assert n % r == 0
    m = n // r
    out = [None] * n
    if not dif:                                           # decimation in time: sub-transforms first
        subs = [fft(d, xs[j::r], sgn, radices[1:], dif) for j in range(r)]
        for k in range(m):
            t = [subs[0][k]] + [c_mulc(d, _tw(sgn, j * k, n), subs[j][k]) for j in range(1, r)]
            y = small_dft(d, t, sgn)
            for p in range(r):
                out[k + m * p] = y[p]
    else:                                                 # decimation in frequency: butterflies first
        cols = []
        for k in range(m):
            y = small_dft(d, [xs[k + m * j] for j in range(r)], sgn)
            cols.append([y[0]] + [c_mulc(d, _tw(sgn, p * k, n), y[p]) for p in range(1, r)])
        for p in range(r):
            sub = fft(d, [cols[k][p] for k in range(m)], sgn, radices[1:], dif)
            for kk in range(m):
                out[r * kk + p] = sub[kk]
    return out


def _tw(sgn, num, den):
    c, s = cis(num, den)
    return (c, sgn * s)


def ktilde(j, n):
    return 2.0 * math.pi * (j if 2 * j < n else j - n) / n


def r2c_network(n, radices, dif):
    """stand-alone DAG of the real-to-complex transform: outputs [Re X_0 .. Re X_h, Im X_1 .. Im X_{h-1}], h = n / 2,
    X_k = sum_j x_j exp(-2 pi i j k / n)."""
    d = Dag(n)
    X = fft(d, [(d.inputs[i], None) for i in range(n)], -1, radices, dif)
    h = n // 2
    assert X[0][1] is None and X[h][1] is None
    return d, [X[k][0] for k in range(h + 1)] + [X[k][1] for k in range(1, h)]


def apply_network(src, src_outs, dst, ins):
    """evaluate the network (src, src_outs) on the values `ins` (signed references in dst): returns the outputs."""
    val = {}
    for nid in range(len(src.kind)):
        k = src.kind[nid]
        if k == "in":
            val[nid] = ins[src.args[nid][0]]
        elif k == "add":
            val[nid] = dst.add(val[src.args[nid][0]], val[src.args[nid][1]])
        elif k == "sub":
            val[nid] = dst.sub(val[src.args[nid][0]], val[src.args[nid][1]])
        else:
            val[nid] = dst.mul(src.args[nid][0], val[src.args[nid][1]])
    return [None if r is None else (dst.mul(r[1], val[r[0]])) for r in src_outs]


def apply_transposed(src, src_outs, dst, ins):
    """the TRANSPOSED linear network (same multiplications, additions run backwards) applied to `ins` (one value per
    output of src): returns one value per input of src.  Used for the complex-to-real transforms: the Hermitian-input
    inverse is, up to weights folded into the spectral multipliers, the transpose of the real-input forward one."""
    acc = {}

    def bump(nid, v):
        acc[nid] = dst.add(acc.get(nid), v)
    for r, v in zip(src_outs, ins):
        if r is not None and v is not None:
            bump(r[0], dst.mul(r[1], v))
    for nid in range(len(src.kind) - 1, -1, -1):
        a = acc.get(nid)
        if a is None:
            continue
        k = src.kind[nid]
        if k == "add":
            bump(src.args[nid][0], a); bump(src.args[nid][1], a)
        elif k == "sub":
            bump(src.args[nid][0], a); bump(src.args[nid][1], dst.neg(a))
        elif k == "mul":
            bump(src.args[nid][1], dst.mul(src.args[nid][0], a))
    return [acc.get(src.inputs[i][0]) for i in range(src.nin)]


def build(n, which, plan):
    """DAG of one codelet.  which = 'inner': inputs x[n] -> outputs a[n], b[n];  'outer': inputs g[n], q[n] -> c[n].
    plan = (radices, dif) of the real-to-complex network; the complex-to-real transforms are its transpose."""
    net, net_outs = r2c_network(n, *plan)
    h = n // 2
    # packed spectrum index: Re X_k -> k (0..h), Im X_k -> h + k (1..h-1)

    def spectral(d, X, first, second):
        """z = weights * (i k X * first + (-k^2) X * second) / n in packed form (transposed-network input)."""
        z = [None] * n
        for k in range(h + 1):
            kt = ktilde(k, n)
            w = 1.0 if k in (0, h) else 2.0
            re = lambda Y: Y[k]
            im = lambda Y: Y[h + k] if 0 < k < h else None
            zr = zi = None
            if second is not None:
                zr = d.mul(-kt * kt * w / n, re(second)); zi = d.mul(-kt * kt * w / n, im(second))
            if first is not None and 0 < k < h:                  # i k (re + i im) = -k im + i k re; Nyquist and 0 dropped
                zr = d.add(zr, d.mul(-kt * w / n, im(first))); zi = d.add(zi, d.mul(kt * w / n, re(first)))
            z[k] = zr
            if 0 < k < h:
                z[h + k] = zi
        return z
    if which == "inner":
        d = Dag(n)
        X = apply_network(net, net_outs, d, d.inputs)
        a = apply_transposed(net, net_outs, d, spectral(d, X, X, None))
        b = apply_transposed(net, net_outs, d, spectral(d, X, None, X))
        return d, [a, b]
    d = Dag(2 * n)
    G = apply_network(net, net_outs, d, d.inputs[:n])
    Q = apply_network(net, net_outs, d, d.inputs[n:])
    c = apply_transposed(net, net_outs, d, spectral(d, G, G, Q))
    return d, [c]


def schedule(d, outs):
    """dead-code elimination, FMA fusion and instruction count.  Returns (ops, stats); ops = list of
    (node, text-builder tuple) in topological order."""
    live = set()
    stack = [r[0] for o in outs for r in o if r is not None]
    while stack:
        n = stack.pop()
        if n in live:
            continue
        live.add(n)
        k = d.kind[n]
        if k in ("add", "sub"):
            stack.extend(d.args[n])
        elif k == "mul":
            stack.append(d.args[n][1])
    # uses of mul nodes that cannot be fused into an add/sub (outputs, or both operands of an add being muls)
    standalone = set()
    fused = {}                                            # add/sub node -> index (0/1) of the operand fused as a multiply
    for o in outs:
        for r in o:
            if r is not None and d.kind[r[0]] == "mul":
                standalone.add(r[0])
    for n in sorted(live):
        if d.kind[n] in ("add", "sub"):
            a, b = d.args[n]
            ma, mb = d.kind[a] == "mul", d.kind[b] == "mul"
            if ma and mb:
                # fuse the one that is not needed on its own anyway
                if b in standalone and a not in standalone:
                    fused[n] = 0; standalone.add(b)
                else:
                    fused[n] = 1; standalone.add(a)
            elif mb:
                fused[n] = 1
            elif ma:
                fused[n] = 0
    nadd = nmul = nfma = 0
    order = []
    depth = {}
    for n in sorted(live):
        k = d.kind[n]
        if k == "in":
            depth[n] = 0
        elif k == "mul":
            depth[n] = depth[d.args[n][1]] + (1 if n in standalone else 0)
        else:
            depth[n] = 1 + max(depth[d.args[n][0]], depth[d.args[n][1]])
    for n in sorted(live, key=lambda v: (depth[v], v)):
        k = d.kind[n]
        if k == "in":
            continue
        if k == "mul":
            if n in standalone:
                nmul += 1; order.append(n)
            continue
        if n in fused:
            nfma += 1
        else:
            nadd += 1
        order.append(n)
    nneg = sum(1 for o in outs for r in o if r is not None and r[1] < 0)
    return order, fused, standalone, dict(add=nadd, mul=nmul, fma=nfma, neg=nneg, total=nadd + nmul + nfma + nneg)


def plans(n):
    """candidate factorisation orders (radix per level) x DIT / DIF of the real-to-complex network."""
    def orders(m):
        if m == 1:
            return [()]
        res = []
        for r in (4, 2, 3, 5):
            if m % r == 0:
                res += [(r,) + t for t in orders(m // r)]
        return res
    for o in orders(n):
        for dif in (False, True):
            yield o, dif


def dense_ops(n):
    """D and D2 (unit spacing) from the defining sums, in long double."""
    j = np.arange(n)
    k = np.array([ktilde(int(x), n) for x in j], dtype=np.longdouble)
    ph = 2.0 * np.pi * np.outer(j, j).astype(np.longdouble) / n
    Fr, Fi = np.cos(ph), -np.sin(ph)                      # F = Fr + i Fi (forward, e^{-ikx})
    k1 = k.copy(); k1[n // 2] = 0.0
    # D = (1/n) conj(F)^T diag(i k) F, real part (imaginary part vanishes)
    D1 = -(Fr.T @ (k1[:, None] * Fi) - Fi.T @ (k1[:, None] * Fr)) / n
    D2 = (Fr.T @ ((-k * k)[:, None] * Fr) + Fi.T @ ((-k * k)[:, None] * Fi)) / n
    return D1, D2


def verify(n, which, d, outs):
    D1, D2 = dense_ops(n)
    def mat(o):
        return np.array([np.zeros(d.nin, dtype=np.longdouble) if r is None else d.valform(r) for r in o])
    if which == "inner":
        e1 = np.abs(mat(outs[0]) - D1).max(); e2 = np.abs(mat(outs[1]) - D2).max()
        return float(max(e1, e2))
    want = np.concatenate([D1, D2], axis=1)
    return float(np.abs(mat(outs[0]) - want).max())


def best(n, which, budget=None):
    bestv = None
    for plan in plans(n):
        d, outs = build(n, which, plan)
        order, fused, standalone, st = schedule(d, outs)
        if bestv is None or st["total"] < bestv[0]["total"]:
            bestv = (st, plan, d, outs, order, fused, standalone)
    st, plan, d, outs, order, fused, standalone = bestv
    err = verify(n, which, d, outs)
    assert err < 1e-13 * n, (n, which, err)
    return bestv + (err,)


def cnum(c):
    return repr(float(c))


def emit(n, which, res):
    st, plan, d, outs, order, fused, standalone, err = res
    innames = (["x"], n) if which == "inner" else (["g", "q"], n)

    def name(nid):
        if d.kind[nid] == "in":
            i = d.args[nid][0]
            return f"{innames[0][i // n]}[{i % n}]"
        return f"t{nid}"
    lines = []
    for nid in order:
        k = d.kind[nid]
        if k == "mul":
            c, a = d.args[nid]
            lines.append(f"const double t{nid} = {cnum(c)} * {name(a)};")
            continue
        a, b = d.args[nid]
        sb = "+" if k == "add" else "-"
        if nid in fused:
            if fused[nid] == 1:                           # a (+|-) c * y
                c, y = d.args[b]
                c = c if k == "add" else -c
                lines.append(f"const double t{nid} = fma({cnum(c)}, {name(y)}, {name(a)});")
            else:                                         # c * y (+|-) b
                c, y = d.args[a]
                lines.append(f"const double t{nid} = fma({cnum(c)}, {name(y)}, {'' if k == 'add' else '-'}{name(b)});")
        else:
            lines.append(f"const double t{nid} = {name(a)} {sb} {name(b)};")
    outnames = ["a", "b"] if which == "inner" else ["c"]
    for o, on in zip(outs, outnames):
        for i, r in enumerate(o):
            if r is None:
                lines.append(f"{on}[{i}] = 0.0;")
            else:
                lines.append(f"{on}[{i}] = {'-' if r[1] < 0 else ''}{name(r[0])};")
    return lines


HEADER = '''// line_codelets.cuh -- GENERATED by gen_codelets.py (do not edit; the build regenerates it).
// Straight-line fp64 code for the lattice line operators D (first derivative, Nyquist mode zeroed) and D2 (second
// derivative) of PAPER.md Eqs. 49-50 on a periodic line of N REAL samples with unit spacing, as real-input FFTs:
//   LineCodelet<N>::inner(x, a, b):   a = D x,  b = D2 x
//   LineCodelet<N>::outer(g, q, c):   c = D g + D2 q
// The instruction counts (DADD / DMUL / DFMA) are listed per codelet; 5 N log2 N / 2 per real transform is the
// nominal FFT count of SURVEY.md 8(d).
#pragma once

template <int N> struct LineCodelet;
'''


def generate(path, sizes=LINE_SIZES, verbose=False):
    parts = [HEADER]
    table = []
    for n in sizes:
        ri = best(n, "inner")
        ro = best(n, "outer")
        nominal = 2.5 * n * math.log2(n)
        table.append((n, ri[0], ro[0], nominal))
        parts.append(f"// N = {n}: inner {ri[0]} (3 real transforms, nominal {3 * nominal:.0f} flop), plan {ri[1]}, "
                     f"max |error of the operator matrix| {ri[7]:.1e}")
        parts.append(f"//         outer {ro[0]} plan {ro[1]}, {ro[7]:.1e}")
        parts.append(f"template <> struct LineCodelet<{n}> {{")
        parts.append(f"    static constexpr int OPS_INNER = {ri[0]['total']}, OPS_OUTER = {ro[0]['total']};")
        parts.append(f"    static __device__ __forceinline__ void inner(const double (&x)[{n}], double (&a)[{n}], double (&b)[{n}])\n    {{")
        parts += ["        " + l for l in emit(n, "inner", ri)]
        parts.append("    }")
        parts.append(f"    static __device__ __forceinline__ void outer(const double (&g)[{n}], const double (&q)[{n}], double (&c)[{n}])\n    {{")
        parts += ["        " + l for l in emit(n, "outer", ro)]
        parts.append("    }")
        parts.append("};\n")
        if verbose:
            print(f"N={n}: inner {ri[0]} outer {ro[0]}  nominal/transform {nominal:.0f}", file=sys.stderr)
    text = "\n".join(parts) + "\n"
    tmp = path + f".tmp{os.getpid()}"
    with open(tmp, "w") as f:
        f.write(text)
    os.replace(tmp, path)
    return table


if __name__ == "__main__":
    out = sys.argv[1] if len(sys.argv) > 1 else os.path.join(os.path.dirname(os.path.abspath(__file__)), "line_codelets.cuh")
    generate(out, verbose=True)
