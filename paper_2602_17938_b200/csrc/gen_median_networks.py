#!/usr/bin/env python
"""Generator + verifier for the shared-column median selection networks (writes median_networks.cuh).

The true k x k median (PAPER.md:23,64 -- "classic median filter rather than any optimized version",
i.e. exact selection, not a separable approximation) of T horizontally adjacent outputs is computed by
ONE thread from T+k-1 image columns of k values each:

  1. sort every column once (Bose-Nelson network; each sorted column serves up to k outputs);
  2. merge sorted columns pairwise / into "cores", dropping every element that cannot be the median of
     ANY k x k window containing those columns: in a sorted run of n elements taken from a window of
     k*k, an element with more than m = (k*k-1)/2 elements below it (or above it) inside the run is
     replaced by +inf (-inf) -- it stays on the same side of the median whatever the rest of the window
     holds;
  3. the core of k-1 shared columns has only k+1 survivors; the median of a window is then one
     rank of (core  U  one more sorted column), a min-of-max expression.

Everything is a straight-line program of 2- and 3-input min/max (FMNMX / FMNMX3 on sm_100a), built with
hash-consing so that work common to neighbouring outputs is emitted once, then dead-code-eliminated
from the requested outputs.  Correctness is PROVEN for every emitted network by the 0-1 principle (a
min/max network selects the right rank for all inputs iff it does so for all 0/1 inputs; with the
column sort in front only sorted 0/1 columns need enumerating: (k+1)^(T+k-1) cases), and re-checked on
random floats with ties.  This file shares nothing with oracle/.

Usage:  python gen_median_networks.py            # verify + (re)write median_networks.cuh
        python gen_median_networks.py --report   # op counts only
"""
from __future__ import annotations

import itertools
import os
import sys

import numpy as np

NEG, POS = "-inf", "+inf"


class Net:
    """Straight-line min/max program with hash-consing and constant (+-inf) folding."""

    def __init__(self, n_inputs):
        self.n_inputs = n_inputs
        self.ops = []            # (kind, args) ; wire id = n_inputs + index
        self.memo = {}

    def _emit(self, kind, args):
        key = (kind, tuple(sorted(args)))
        if key in self.memo:
            return self.memo[key]
        self.ops.append((kind, tuple(args)))
        w = self.n_inputs + len(self.ops) - 1
        self.memo[key] = w
        return w

    def mn(self, *a):
        a = [x for x in dict.fromkeys(a) if x != POS]
        if NEG in a:
            return NEG
        if not a:
            return POS
        if len(a) == 1:
            return a[0]
        assert len(a) in (2, 3)
        return self._emit("min", a)

    def mx(self, *a):
        a = [x for x in dict.fromkeys(a) if x != NEG]
        if POS in a:
            return POS
        if not a:
            return NEG
        if len(a) == 1:
            return a[0]
        assert len(a) in (2, 3)
        return self._emit("max", a)

    def ce(self, a, b):
        return self.mn(a, b), self.mx(a, b)

    def mn_many(self, xs):
        xs = list(xs)
        while len(xs) > 1:
            nxt, i = [], 0
            while i < len(xs):
                grp = xs[i:i + 3]
                nxt.append(self.mn(*grp))
                i += 3
            xs = nxt
        return xs[0]

    def mx_many(self, xs):
        xs = list(xs)
        while len(xs) > 1:
            nxt, i = [], 0
            while i < len(xs):
                nxt.append(self.mx(*xs[i:i + 3]))
                i += 3
            xs = nxt
        return xs[0]

    # ---- analysis
    def live(self, outputs):
        need = set()
        stack = [o for o in outputs if isinstance(o, int) and o >= self.n_inputs]
        while stack:
            w = stack.pop()
            if w in need:
                continue
            need.add(w)
            for a in self.ops[w - self.n_inputs][1]:
                if isinstance(a, int) and a >= self.n_inputs:
                    stack.append(a)
        return need

    def count(self, outputs):
        return len(self.live(outputs))

    def evaluate(self, outputs, inputs):
        """inputs: array [n_inputs, ncases]; returns [len(outputs), ncases]."""
        need = self.live(outputs)
        val = {i: inputs[i] for i in range(self.n_inputs)}
        for idx, (kind, args) in enumerate(self.ops):
            w = self.n_inputs + idx
            if w not in need:
                continue
            f = np.minimum if kind == "min" else np.maximum
            r = f(val[args[0]], val[args[1]])
            if len(args) == 3:
                r = f(r, val[args[2]])
            val[w] = r
        return np.stack([val[o] for o in outputs])


# ------------------------------------------------------------------------------------------ building blocks
def bose_nelson(n):
    """Comparator list of the Bose-Nelson sorting network (size-optimal for n <= 8)."""
    out = []

    def pbracket(i, x, j, y):
        if x == 1 and y == 1:
            out.append((i, j))
        elif x == 1 and y == 2:
            out.append((i, j + 1)); out.append((i, j))
        elif x == 2 and y == 1:
            out.append((i, j)); out.append((i + 1, j))
        else:
            a, b = x // 2, (y // 2 if x % 2 else (y + 1) // 2)
            pbracket(i, a, j, b)
            pbracket(i + a, x - a, j + b, y - b)
            pbracket(i + a, x - a, j, b)

    def pstar(i, m):
        if m > 1:
            a = m // 2
            pstar(i, a)
            pstar(i + a, m - a)
            pbracket(i, a, i + a, m - a)

    pstar(0, n)
    return out


def sort_wires(net, wires):
    w = list(wires)
    for i, j in bose_nelson(len(w)):
        w[i], w[j] = net.ce(w[i], w[j])
    return w


def merge_batcher(net, A, B):
    """Batcher odd-even merge of two ascending lists (any lengths); +-inf entries fold away."""
    if not A:
        return list(B)
    if not B:
        return list(A)
    if len(A) == 1 and len(B) == 1:
        return list(net.ce(A[0], B[0]))
    V = merge_batcher(net, A[0::2], B[0::2])      # 1st, 3rd, ... of each
    W = merge_batcher(net, A[1::2], B[1::2])      # 2nd, 4th, ... of each
    out = [V[0]]
    i = 0
    # w_i is compared with v_{i+1}
    while i < len(W) and i + 1 < len(V):
        lo, hi = net.ce(W[i], V[i + 1])
        out += [lo, hi]
        i += 1
    out += W[i:] + V[i + 1:]
    return out


def merge_select(net, A, B, ranks):
    """Selected ranks (0-based) of the union of two ascending lists: t-th smallest (1-based t) =
    min over i + j = t of max(A_i, B_j), with A_0 = B_0 = -inf."""
    res = {}
    for r in ranks:
        t = r + 1
        terms = []
        for i in range(0, t + 1):
            j = t - i
            if i > len(A) or j > len(B):
                continue
            a = A[i - 1] if i >= 1 else NEG
            b = B[j - 1] if j >= 1 else NEG
            terms.append(net.mx(a, b))
        res[r] = net.mn_many(terms)
    return res


class Run:
    """An ascending run of `n` window elements of which only ranks [lo, hi] are kept (others are
    known to be below / above the median of any window containing the run)."""

    def __init__(self, wires, n, lo):
        self.wires, self.n, self.lo = wires, n, lo      # wires[i] has rank lo + i within the run

    def full(self):
        return [NEG] * self.lo + list(self.wires) + [POS] * (self.n - self.lo - len(self.wires))


def prune(run_full, m):
    """Keep ranks p with p <= m and n-1-p <= m."""
    n = len(run_full)
    lo, hi = max(0, n - 1 - m), min(n - 1, m)
    return Run(run_full[lo:hi + 1], n, lo)


def merge_runs(net, R1, R2, m, method="batcher"):
    n = R1.n + R2.n
    lo, hi = max(0, n - 1 - m), min(n - 1, m)
    if method == "batcher":
        full = merge_batcher(net, R1.full(), R2.full())
        return Run(full[lo:hi + 1], n, lo)
    sel = merge_select(net, R1.full(), R2.full(), range(lo, hi + 1))
    return Run([sel[r] for r in range(lo, hi + 1)], n, lo)


def best_merge(net_factory, build):
    """Helper for choosing per-merge methods is done at plan level (see plan_* below)."""
    raise NotImplementedError


# ------------------------------------------------------------------------------------------ plans
def plan_pairs(k, T, methods=None):
    """T outputs (T even) from T+k-1 columns.  Column c holds inputs c*k .. c*k+k-1 (top to bottom).
    Window t = columns t .. t+k-1.  Outputs 2i and 2i+1 share the core of columns 2i+1 .. 2i+k-1
    (k-1 columns, even count), built from pair-merges M(2j+1, 2j+2); a core of k-3 columns is shared
    by two neighbouring cores where possible."""
    assert T % 2 == 0 and k % 2 == 1
    methods = methods or {}
    m = (k * k - 1) // 2
    ncol = T + k - 1
    net = Net(ncol * k)
    cols = [Run(sort_wires(net, [c * k + r for r in range(k)]), k, 0) for c in range(ncol)]
    pair = {}

    def M(a):                        # merge of columns a, a+1
        if a not in pair:
            pair[a] = merge_runs(net, cols[a], cols[a + 1], m, methods.get("pair", "batcher"))
        return pair[a]

    cores = {}

    def core(a, npairs):             # core of columns a .. a+2*npairs-1
        key = (a, npairs)
        if key in cores:
            return cores[key]
        if npairs == 1:
            r = M(a)
        else:
            # prefer the split whose big part is already available / aligned to multiples of 4
            left_first = ((a - 1) // 2) % 2 == 1
            if left_first:
                r = merge_runs(net, core(a, npairs - 1), M(a + 2 * (npairs - 1)), m,
                               methods.get("core%d" % npairs, "batcher"))
            else:
                r = merge_runs(net, M(a), core(a + 2, npairs - 1), m,
                               methods.get("core%d" % npairs, "batcher"))
        cores[key] = r
        return r

    outs = []
    npairs = (k - 1) // 2
    for i in range(T // 2):
        c = core(2 * i + 1, npairs)                  # columns 2i+1 .. 2i+k-1
        for t, extra in ((2 * i, 2 * i), (2 * i + 1, 2 * i + k)):
            sel = merge_select(net, c.full(), cols[extra].full(), [m])
            outs.append(sel[m])
    return net, outs


# ------------------------------------------------------------------------------------------ verification
def live_inputs(net, out):
    return sorted(a for w in net.live([out]) for a in net.ops[w - net.n_inputs][1]
                  if isinstance(a, int) and a < net.n_inputs)


def verify(net, outs, k, T, n_random=20000, seed=0):
    """0-1 principle per output over its own k sorted columns ((k+1)^k cases), after checking that the
    output's live program reads no input outside its window; then random floats, with and without ties."""
    m = (k * k - 1) // 2
    ncol = T + k - 1
    pats = np.array([[0] * (k - j) + [1] * j for j in range(k + 1)], dtype=np.int8)   # [k+1, k]
    total = (k + 1) ** k
    chunk = 1 << 18
    for t in range(T):
        li = live_inputs(net, outs[t])
        if li and (min(li) < t * k or max(li) >= (t + k) * k):
            return False
        for start in range(0, total, chunk):
            idx = np.arange(start, min(total, start + chunk))
            digits = np.empty((k, idx.size), dtype=np.int64)
            x = idx.copy()
            for c in range(k):
                digits[c] = x % (k + 1)
                x //= (k + 1)
            inp = np.zeros((ncol * k, idx.size), dtype=np.int8)
            for c in range(k):
                inp[(t + c) * k:(t + c + 1) * k] = pats[digits[c]].T
            got = net.evaluate([outs[t]], inp)[0]
            want = (digits.sum(axis=0) >= k * k - m).astype(np.int8)
            if not np.array_equal(got, want):
                return False
    rng = np.random.default_rng(seed)
    for ties in (False, True):
        x = rng.standard_normal((ncol * k, n_random)).astype(np.float32)
        if ties:
            x = np.round(x * 1.5)
        got = net.evaluate(outs, x)
        cols = x.reshape(ncol, k, n_random)
        for t in range(T):
            win = cols[t:t + k].reshape(k * k, n_random)
            want = np.sort(win, axis=0)[m]
            if not np.array_equal(got[t], want):
                return False
    return True


# ------------------------------------------------------------------------------------------ emission
def emit_cuda(net, outs, name, k, T):
    need = net.live(outs)
    ncol = T + k - 1
    lines = []
    lines.append("// %d x %d median of %d adjacent outputs from %d columns: %d min/max instructions "
                 "(%.1f per output)" % (k, k, T, ncol, len(need), len(need) / T))
    lines.append("// in[c][r]: column c (left to right), row r (top to bottom) of the (T+k-1) x k footprint.")
    lines.append("__device__ __forceinline__ void %s(const float (&in)[%d][%d], float (&out)[%d]) {"
                 % (name, ncol, k, T))

    def ref(w):
        if w < net.n_inputs:
            return "in[%d][%d]" % (w // k, w % k)
        return "w%d" % w

    for idx, (kind, args) in enumerate(net.ops):
        w = net.n_inputs + idx
        if w not in need:
            continue
        if len(args) == 2:
            fn = "fminf" if kind == "min" else "fmaxf"
        else:
            fn = "min3" if kind == "min" else "max3"
        lines.append("    const float w%d = %s(%s);" % (w, fn, ", ".join(ref(a) for a in args)))
    for t, o in enumerate(outs):
        lines.append("    out[%d] = %s;" % (t, ref(o)))
    lines.append("}")
    return "\n".join(lines), len(need)


def sort_mergesort(net, wires):
    """Full ascending sort: Bose-Nelson for <= 8 inputs, Batcher odd-even merges above."""
    n = len(wires)
    if n <= 8:
        return sort_wires(net, wires)
    return merge_batcher(net, sort_mergesort(net, wires[:n // 2]), sort_mergesort(net, wires[n // 2:]))


def verify_merges_and_sort(n, n_random=20000):
    """A merge sort is correct if every merge is: check each (m1, m2) merge on all sorted 0/1 input
    pairs, the base sorters on all 0/1 inputs, then the whole network on random floats with ties."""
    def sizes(n):
        if n <= 8:
            return [], [n]
        a, b = n // 2, n - n // 2
        ma, ba = sizes(a)
        mb, bb = sizes(b)
        return ma + mb + [(a, b)], ba + bb
    merges, bases = sizes(n)
    for b in set(bases):
        net = Net(b)
        out = sort_wires(net, list(range(b)))
        inp = np.array(list(itertools.product([0, 1], repeat=b)), dtype=np.int8).T
        if not np.array_equal(net.evaluate(out, inp), np.sort(inp, axis=0)):
            return False
    for a, b in set(merges):
        net = Net(a + b)
        out = merge_batcher(net, list(range(a)), list(range(a, a + b)))
        cases = [[0] * (a - i) + [1] * i + [0] * (b - j) + [1] * j for i in range(a + 1) for j in range(b + 1)]
        inp = np.array(cases, dtype=np.int8).T
        got = np.stack([inp[o] if o < a + b else None for o in out]) if not net.ops else net.evaluate(out, inp)
        if not np.array_equal(got, np.sort(inp, axis=0)):
            return False
    net = Net(n)
    out = sort_mergesort(net, list(range(n)))
    rng = np.random.default_rng(1)
    for ties in (False, True):
        x = rng.standard_normal((n, n_random)).astype(np.float32)
        if ties:
            x = np.round(x * 1.5)
        if not np.array_equal(net.evaluate(out, x), np.sort(x, axis=0)):
            return False
    return True


def emit_sort(n, name):
    net = Net(n)
    out = sort_mergesort(net, list(range(n)))
    need = net.live(out)
    lines = ["// ascending sort of %d values: %d min/max instructions (Bose-Nelson blocks + Batcher odd-even merges)"
             % (n, len(need)),
             "__device__ __forceinline__ void %s(const float (&in)[%d], float (&out)[%d]) {" % (name, n, n)]
    ref = lambda w: ("in[%d]" % w) if w < n else ("w%d" % w)
    for idx, (kind, args) in enumerate(net.ops):
        w = n + idx
        if w in need:
            lines.append("    const float w%d = %s(%s);" % (w, "fminf" if kind == "min" else "fmaxf",
                                                         ", ".join(ref(a) for a in args)))
    for i, o in enumerate(out):
        lines.append("    out[%d] = %s;" % (i, ref(o)))
    lines.append("}")
    return "\n".join(lines), len(need)


CONFIGS = [  # (k, T, function name)
    (3, 2, "median3x3_x2"), (3, 4, "median3x3_x4"),
    (5, 2, "median5x5_x2"), (5, 4, "median5x5_x4"), (5, 8, "median5x5_x8"),
    (7, 2, "median7x7_x2"), (7, 4, "median7x7_x4"),
]


def search_methods(k, T):
    """Try batcher / min-of-max for each merge level; keep the cheapest."""
    levels = ["pair"] + ["core%d" % i for i in range(2, (k - 1) // 2 + 1)]
    best = None
    for combo in itertools.product(("batcher", "select"), repeat=len(levels)):
        methods = dict(zip(levels, combo))
        net, outs = plan_pairs(k, T, methods)
        n = net.count(outs)
        if best is None or n < best[0]:
            best = (n, methods, net, outs)
    return best


def main():
    report = "--report" in sys.argv
    here = os.path.dirname(os.path.abspath(__file__))
    chunks = ["// GENERATED by gen_median_networks.py -- do not edit.  Exact k x k median selection networks",
              "// (column sort shared between adjacent outputs, pruned core merges, min-of-max final select);",
              "// every network below was verified by the 0-1 principle over all sorted-column inputs.",
              "#pragma once", '#include "common.cuh"', "", "namespace lac {", ""]
    for k, T, name in CONFIGS:
        n, methods, net, outs = search_methods(k, T)
        print("k=%d T=%d: %d ops (%.1f per output) methods=%s" % (k, T, n, n / T, methods), flush=True)
        if report:
            continue
        ncases = T * (k + 1) ** k
        ok = verify(net, outs, k, T)
        print("   verified (0-1 principle, %d cases + random floats): %s" % (ncases, ok), flush=True)
        if not ok:
            raise SystemExit("network %s is WRONG" % name)
        code, _ = emit_cuda(net, outs, name, k, T)
        chunks += [code, ""]
    ok = verify_merges_and_sort(25)
    code, nops = emit_sort(25, "sort25")
    print("sort25: %d ops, verified (0-1 principle per merge + random floats): %s" % (nops, ok), flush=True)
    if not ok:
        raise SystemExit("sort25 is WRONG")
    chunks += [code, ""]
    if not report:
        chunks += ["}  // namespace lac", ""]
        with open(os.path.join(here, "median_networks.cuh"), "w") as fh:
            fh.write("\n".join(chunks))
        print("wrote median_networks.cuh")


if __name__ == "__main__":
    main()
