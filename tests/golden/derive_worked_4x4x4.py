"""Exact-rational hand evaluation of the 4^3 worked example (pin I13).

Independent of oracle/ and of the CUDA path: python `fractions` for everything rational
(differences, q+ = (nabla+)^2, q- = (nabla-)^2, cut-off), 40-digit `decimal` for the square
roots.  Follows PAPER.md eq. 3 (line 25), eq. 4-5 (30-35), eq. 6 (43), eq. 7 (48), eq. 11 (67),
eq. 12-13 (76-82) with readings R1-R6, R10, R12 of DESIGN.md.

Set-up: grid 4x4x4, dx = 1, gamma = 3, beta = 3/2, dt = 1/2, dtau = 1/2 (deliberately not
CFL-safe; it only pins arithmetic).  phi0(i,j,k) = (3/2)i - (1/2)j^2 + (1/4)jk + k - 9/4;
F(i,j,k) = 1 if (i+j+k) even else -1/2.  All phi0 are dyadic, so q+- are exact rationals.

`python tests/golden/derive_worked_4x4x4.py` prints exactly what
tests/golden/worked_4x4x4.txt stores (the test re-runs it and compares).
"""
from decimal import Decimal, getcontext
from fractions import Fraction as Fr

getcontext().prec = 40
n = 4
dx, gamma, beta, dt, dtau = Fr(1), Fr(3), Fr(3, 2), Fr(1, 2), Fr(1, 2)
PTS = [(i, j, k) for k in range(n) for j in range(n) for i in range(n)]
phi = {(i, j, k): Fr(3, 2) * i - Fr(1, 2) * j * j + Fr(1, 4) * j * k + k - Fr(9, 4) for (i, j, k) in PTS}
F = {(i, j, k): Fr(1) if (i + j + k) % 2 == 0 else Fr(-1, 2) for (i, j, k) in PTS}
AXES = [(1, 0, 0), (0, 1, 0), (0, 0, 1)]


def cl(v):
    return min(max(v, 0), n - 1)


def at(f, i, j, k):                      # edge replicate (R3)
    return f[(cl(i), cl(j), cl(k))]


def dec(fr):
    return Decimal(fr.numerator) / Decimal(fr.denominator)


def one_sided(f, p, h):                  # [(D-x, D+x), (D-y, D+y), (D-z, D+z)]   (R1)
    i, j, k = p
    c = f[p]
    return [((c - at(f, i - e[0], j - e[1], k - e[2])) / h, (at(f, i + e[0], j + e[1], k + e[2]) - c) / h)
            for e in AXES]


def q_pm(D, zero):                       # eq. 4, eq. 5 (squares, before the root)
    qp = sum(max(a, zero) ** 2 + min(b, zero) ** 2 for a, b in D)
    qm = sum(max(b, zero) ** 2 + min(a, zero) ** 2 for a, b in D)
    return qp, qm


def cut(v):                              # eq. 7
    a = abs(v)
    if a <= beta:
        return Fr(1)
    if a <= gamma:
        return (a - gamma) ** 2 * (2 * a + gamma - 3 * beta) / (gamma - beta) ** 3
    return Fr(0)


def face_nb(p):
    for e in AXES:
        for s in (1, -1):
            q = (p[0] + s * e[0], p[1] + s * e[1], p[2] + s * e[2])
            if all(0 <= c < n for c in q):
                yield q


T = {p: abs(phi[p]) < gamma for p in PTS}                            # eq. 6
N = {p: T[p] or any(T[q] for q in face_nb(p)) for p in PTS}          # eq. 11 (R6)


def words(M):                            # R20: word lz, bit ly*8+lx
    return ["0x%08x" % sum(1 << (ly * 8 + lx) for ly in range(n) for lx in range(n) if M[(lx, ly, lz)])
            for lz in range(n)]


# Advance, eq. 3 with eq. 8
bar = {}
for p in PTS:
    if T[p]:
        qp, qm = q_pm(one_sided(phi, p, dx), Fr(0))
        H = dec(max(F[p], Fr(0))) * dec(qp).sqrt() + dec(min(F[p], Fr(0))) * dec(qm).sqrt()
        bar[p] = dec(phi[p]) - dec(dt) * dec(cut(phi[p])) * H
    else:
        bar[p] = dec(phi[p])

# one reinitialisation iteration, eq. 12-13 (R10: |Dd|^2 = q+ if d > 0, q- if d < 0)
d1 = {}
Z = Decimal(0)
for p in PTS:
    if N[p]:
        qp, qm = q_pm(one_sided(bar, p, Decimal(1)), Z)
        c = bar[p]
        qq = qp if c > 0 else (qm if c < 0 else Z)
        den = (c * c + qq * dec(dx) ** 2).sqrt()
        S = c / den if den != 0 else Z
        U = max(S, Z) * (qp.sqrt() - 1) + min(S, Z) * (qm.sqrt() - 1)
        d1[p] = c - dec(dtau) * U
    else:
        d1[p] = bar[p]


def main():
    print("# 4^3 worked example; written by tests/golden/derive_worked_4x4x4.py (exact rationals; see its docstring)")
    print("count T %d" % sum(T.values()))
    print("count N %d" % sum(N.values()))
    print("words T " + " ".join(words(T)))
    print("words N " + " ".join(words(N)))
    for p in [(2, 0, 2), (3, 1, 0), (0, 0, 3), (1, 1, 1), (1, 2, 1), (2, 3, 2)]:
        qp, qm = q_pm(one_sided(phi, p, dx), Fr(0))
        print("point %d %d %d phi %s qp %s qm %s c %s F %s bar %.20e" %
              (p + (phi[p], qp, qm, cut(phi[p]), F[p], bar[p])))
    for p in [(1, 2, 1), (0, 0, 3), (2, 3, 2), (1, 1, 1)]:
        print("reinit %d %d %d d1 %.20e" % (p + (d1[p],)))
    print("sum bar %.20e" % sum(bar.values()))
    print("sum d1 %.20e" % sum(d1.values()))
    # every value, for the element-wise comparison
    for p in PTS:
        print("all %d %d %d %.20e %.20e" % (p + (bar[p], d1[p])))


if __name__ == "__main__":
    main()
