#!/usr/bin/env python
"""Generate butterflies_gen.cuh: straight-line in-register DFTs of R = 2, 4, 8, 16 complex points
written with Blackwell's packed FP32x2 instructions (FADD2 / FFMA2 on (re, im) register pairs).

    python paper_1711_10855_b200/csrc/gen_butterflies.py        # rewrites butterflies_gen.cuh

What is generated is eq.(3) of arXiv:1711.10855 for N = R by the divide and
conquer of PAPER.md line 40, factored R = R1 x R2 (Cooley-Tukey, natural order in and out):

    X[k1 + R1 k2] = sum_{n2} w_R^{n2 k1} w_{R2}^{n2 k2}  sum_{n1} x[R2 n1 + n2] w_{R1}^{n1 k1}

Cost model (sm_100a): one FADD2 / FFMA2 does a complex add, or a complex "a + s*b", in ONE issue
slot; operand swaps (re<->im), per-half negation and scalar broadcast are free operand modifiers
(SASS: .F32x2.LO_HI, .NP/.PN, .F32).  So
  * multiplication by +-i is never executed: it is a pending rotation folded into the consumer,
  * a constant twiddle w = c (1 + i t), |t| <= 1 (angles outside +-45 degrees first take out a
    quarter turn) costs ONE FFMA2:  v' = v + t (i v);  the real factor c stays pending and is
    absorbed by the next add, which becomes an FFMA2 with the ratio of the two pending factors.
Every value is tracked as  true = scale * i^rot * reg.  The leader of every add chain (index 0 of
each sub-transform) has scale 1 and rot 0, so the outputs need no fix-up; the generator asserts it.
Radix-16 comes out at 72 packed instructions (64 adds + 8 twiddles) instead of the 168 scalar
flops of the textbook count.
"""
import math
import os

HERE = os.path.dirname(os.path.abspath(__file__))
OUT = os.path.join(HERE, "butterflies_gen.cuh")


class Val:
    __slots__ = ("name", "scale", "rot")

    def __init__(self, name, scale=1.0, rot=0):
        self.name, self.scale, self.rot = name, scale, rot % 4


class Gen:
    def __init__(self):
        self.lines = []
        self.n_tmp = 0
        self.n_ops = 0

    def tmp(self):
        self.n_tmp += 1
        return f"t{self.n_tmp}"

    @staticmethod
    def rot_expr(name, r):
        """expression for i^r * name as a float2 (the compiler folds it into operand modifiers)"""
        r %= 4
        if r == 0:
            return name
        if r == 1:
            return f"make_float2(-{name}.y, {name}.x)"
        if r == 2:
            return f"make_float2(-{name}.x, -{name}.y)"
        return f"make_float2({name}.y, -{name}.x)"

    @staticmethod
    def lit(x):
        return f"{float(x):.9g}f"

    def addsub(self, u, v, sign):
        """true_u + sign * true_v, result carries u's pending scale and rotation."""
        ratio = sign * v.scale / u.scale
        rel = (v.rot - u.rot) % 4
        out = self.tmp()
        self.n_ops += 1
        if abs(abs(ratio) - 1.0) < 1e-12:
            r = rel if ratio > 0 else (rel + 2) % 4
            self.lines.append(f"const float2 {out} = __fadd2_rn({u.name}, {self.rot_expr(v.name, r)});")
        else:
            c = self.lit(ratio)
            self.lines.append(f"const float2 {out} = __ffma2_rn({self.rot_expr(v.name, rel)}, make_float2({c}, {c}), {u.name});")
        return Val(out, u.scale, u.rot)

    def twiddle(self, v, turns):
        """multiply by exp(2 pi i turns)"""
        q = round(turns * 4.0)
        rem = turns - q / 4.0            # in [-1/8, 1/8]
        rot = v.rot + q
        if abs(rem) < 1e-12:
            return Val(v.name, v.scale, rot)
        th = 2.0 * math.pi * rem
        c, t = math.cos(th), math.tan(th)
        out = self.tmp()
        self.n_ops += 1
        if abs(abs(t) - 1.0) < 1e-12:
            r = 1 if t > 0 else 3
            self.lines.append(f"const float2 {out} = __fadd2_rn({v.name}, {self.rot_expr(v.name, r)});")
        else:
            tt = self.lit(t)
            self.lines.append(f"const float2 {out} = __ffma2_rn({self.rot_expr(v.name, 1)}, make_float2({tt}, {tt}), {v.name});")
        return Val(out, v.scale * c, rot)

    def dft(self, xs, sign):
        n = len(xs)
        if n == 1:
            return xs
        if n == 2:
            return [self.addsub(xs[0], xs[1], +1), self.addsub(xs[0], xs[1], -1)]
        if n == 4:
            a0 = self.addsub(xs[0], xs[2], +1)
            a1 = self.addsub(xs[0], xs[2], -1)
            a2 = self.addsub(xs[1], xs[3], +1)
            a3 = self.addsub(xs[1], xs[3], -1)
            a3 = Val(a3.name, a3.scale, a3.rot + sign)   # * (sign i): forward -i, inverse +i
            return [self.addsub(a0, a2, +1), self.addsub(a1, a3, +1), self.addsub(a0, a2, -1), self.addsub(a1, a3, -1)]
        n1 = 4 if n % 4 == 0 and n > 4 else 2
        n2 = n // n1
        # step 1: for each n2, DFT_{n1} over n1 of x[n2_count*n1_idx + n2_idx]
        T = []
        for j2 in range(n2):
            T.append(self.dft([xs[n2 * j1 + j2] for j1 in range(n1)], sign))   # T[j2][k1]
        # twiddle w_n^{j2 k1}
        for j2 in range(n2):
            for k1 in range(n1):
                T[j2][k1] = self.twiddle(T[j2][k1], sign * (j2 * k1) / n)
        out = [None] * n
        for k1 in range(n1):
            Y = self.dft([T[j2][k1] for j2 in range(n2)], sign)               # Y[k2]
            for k2 in range(n2):
                out[k1 + n1 * k2] = Y[k2]
        return out


def emit(R, inverse):
    g = Gen()
    xs = [Val(f"v[{j}]") for j in range(R)]
    ys = g.dft(xs, +1 if inverse else -1)
    body = list(g.lines)
    fix = 0
    outs = []
    for k, y in enumerate(ys):
        if abs(y.scale - 1.0) < 1e-9:
            outs.append(f"v[{k}] = {Gen.rot_expr(y.name, y.rot)};")
        else:
            fix += 1
            c = Gen.lit(y.scale)
            outs.append(f"v[{k}] = __fmul2_rn({Gen.rot_expr(y.name, y.rot)}, make_float2({c}, {c}));")
    assert fix == 0, f"radix {R}: {fix} outputs need a scale fix-up"
    name = f"dft{R}_{'inv' if inverse else 'fwd'}"
    src = [f"// {R}-point {'inverse (conjugate twiddles, unnormalised)' if inverse else 'forward'} DFT, "
           f"{g.n_ops} packed instructions",
           f"__device__ __forceinline__ void {name}(float2 *v)", "{"]
    src += ["    " + l for l in body]
    src += ["    " + l for l in outs]
    src += ["}", ""]
    return "\n".join(src), g.n_ops


def main():
    parts = ["// butterflies_gen.cuh -- GENERATED by gen_butterflies.py; do not edit.",
             "// In-register DFTs (eq.(3), PAPER.md line 35) in packed FP32x2 form; see the generator's docstring.",
             "#pragma once", "#include <cuda_runtime.h>", "", "namespace fdas {", ""]
    counts = {}
    for R in (2, 4, 8, 16):
        for inv in (False, True):
            s, n = emit(R, inv)
            parts.append(s)
            counts[R] = n
    parts.append("} // namespace fdas")
    with open(OUT, "w") as f:
        f.write("\n".join(parts) + "\n")
    print("wrote", OUT, counts)


if __name__ == "__main__":
    main()
