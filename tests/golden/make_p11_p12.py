"""Writes p11_3d_exact.txt and p12_src_exact.txt: exact-rational two-level examples for the 3-D reading
(R-3D) and for the level with a source term and moving boundary values (R-N3).

Every value is the exact solution (Fractions, Gaussian elimination) of the IMPLICIT statement of a level
assembled node by node in tests/dense_ref.py -- never the closed forms, never oracle/, never the CUDA path.

    python tests/golden/make_p11_p12.py
"""
import os
import sys
from fractions import Fraction as F

HERE = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, os.path.dirname(HERE))
import dense_ref as D  # noqa: E402


def fr(v):
    return " ".join(str(x) for x in v)


def level_3d(u, n, r, phase, bc):
    A, B, c = D.system_3d(n, n, n, F(r), phase, bc, num=F)
    rhs = [sum(B[i][j] * u[j] for j in range(len(u)) if B[i][j] != 0) + c[i] for i in range(len(u))]
    return D.solve_exact(A, rhs)


def level_src(u, r, k, phase, bo, bn, s):
    n = len(u)
    side = D.classes_1d(n, k, phase)
    r = F(r)
    A = [[F(0)] * n for _ in range(n)]
    rhs = [F(0)] * n
    for i in range(1, n + 1):
        A[i - 1][i - 1] = 1 + r
        rhs[i - 1] = (1 - r) * u[i - 1] + s[i - 1]
        jn, jo = i + side[i], i - side[i]
        if jn in (0, n + 1):
            rhs[i - 1] += r * (bn[0] if jn == 0 else bn[1])
        else:
            A[i - 1][jn - 1] -= r
        rhs[i - 1] += r * ((bo[0] if jo == 0 else bo[1]) if jo in (0, n + 1) else u[jo - 1])
    return D.solve_exact(A, rhs)


def main():
    with open(os.path.join(HERE, "p11_3d_exact.txt"), "w") as f:
        f.write("# N r ; bc x_lo x_hi y_lo y_hi z_lo z_hi ; U0 [k][j][i] ; level 1 (phase 0) ; level 2 (phase 1)\n")
        f.write("# DESIGN.md reading R-3D (PAPER.md is silent on 3-D: :134, :228); written by make_p11_p12.py\n")
        for n, r, bc in ((2, 1, (0,) * 6), (2, 2, (1, 0, 0, 3, 0, 2)), (3, 1, (0, 1, 2, 0, 1, 0))):
            u0 = [F(v) for v in range(1, n ** 3 + 1)]
            bcf = tuple(F(b) for b in bc)
            u1 = level_3d(u0, n, r, 0, bcf)
            u2 = level_3d(u1, n, r, 1, bcf)
            f.write("%d %s ; %s ; %s ; %s ; %s\n" % (n, r, fr(bc), fr(u0), fr(u1), fr(u2)))
    with open(os.path.join(HERE, "p12_src_exact.txt"), "w") as f:
        f.write("# k r ; lo(t0) lo(t1) lo(t2) ; hi(t0) hi(t1) hi(t2) ; U0 ; s of level 1 ; s of level 2 ; level 1 (phase 0) ; level 2 (phase 1)\n")
        f.write("# DESIGN.md reading R-N3 (the paper has neither source nor moving boundaries, PAPER.md:57-61); written by make_p11_p12.py\n")
        for k, r, n in ((1, 2, 4), (1, 1, 5), (2, 1, 6)):
            u0 = [F(v) for v in range(1, n + 1)]
            lo = [F(1), F(3, 2), F(2)]
            hi = [F(-1), F(0), F(1, 2)]
            s1 = [F(i, 4) for i in range(1, n + 1)]
            s2 = [F(-i, 8) for i in range(1, n + 1)]
            u1 = level_src(u0, r, k, 0, (lo[0], hi[0]), (lo[1], hi[1]), s1)
            u2 = level_src(u1, r, k, 1, (lo[1], hi[1]), (lo[2], hi[2]), s2)
            f.write("%d %s ; %s ; %s ; %s ; %s ; %s ; %s ; %s\n" % (k, r, fr(lo), fr(hi), fr(u0), fr(s1), fr(s2), fr(u1), fr(u2)))


if __name__ == "__main__":
    main()
