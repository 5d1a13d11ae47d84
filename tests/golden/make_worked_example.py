"""Writes tests/golden/worked_example.json: the worked example of SURVEY.md 8(c).4, recomputed with
Python big integers only (no oracle, no CUDA, no numpy) and by routes that differ from the oracle's:

  nodes          pow(y, e, p) products                                   (eq. (3))
  master poly    coefficients by Vieta: elementary symmetric sums over subsets
  probe values   v_{j,s} = sum_i a_i(c_j) m_i^s from the planted coefficient polynomials (L60)
  den            prod_{j != i} (m_i - m_j)                               (reading G15)
  solved c       Gauss-Jordan over Z/pZ on the t x t system              (O(t^3))
  newton rows    divided differences by the recursive definition f[x_a..x_b] (eq. (1))

The paper prints no numeric example (its only numbers are timings); this file is the stand-in pin.
Run:  python tests/golden/make_worked_example.py
"""
import itertools
import json
import math
import os


def solve_mod(A, b, p):
    n = len(A)
    A = [row[:] + [bi] for row, bi in zip(A, b)]
    for c in range(n):
        piv = next(r for r in range(c, n) if A[r][c] % p)
        A[c], A[piv] = A[piv], A[c]
        inv = pow(A[c][c], -1, p)
        A[c] = [x * inv % p for x in A[c]]
        for r in range(n):
            if r != c and A[r][c]:
                f = A[r][c]
                A[r] = [(x - f * y) % p for x, y in zip(A[r], A[c])]
    return [A[i][n] for i in range(n)]


def divided_difference(xs, fs, a, b, p):
    if a == b:
        return fs[a] % p
    num = divided_difference(xs, fs, a + 1, b, p) - divided_difference(xs, fs, a, b - 1, p)
    return num * pow(xs[b] - xs[a], -1, p) % p


def case(p, anchors, samples):
    E = [(0, 0), (1, 0), (0, 2), (2, 1)]
    planted = [[5, 0, 1], [7, 3, 0], [0, 0, 9], [1, 1, 1]]  # per term: coefficients of x_3^0..x_3^2
    t, B = len(E), len(samples)
    nodes = [pow(anchors[0], e[0], p) * pow(anchors[1], e[1], p) % p for e in E]
    M = []
    for l in range(t + 1):  # coefficient of z^l = (-1)^(t-l) e_{t-l}(nodes)
        e = sum(math.prod(s) for s in itertools.combinations(nodes, t - l))
        M.append((-1) ** (t - l) * e % p)
    a_at = [[sum(c * pow(cj, d, p) for d, c in enumerate(planted[i])) % p for i in range(t)] for cj in samples]
    vals = [[sum(a_at[j][i] * pow(nodes[i], s, p) for i in range(t)) % p for s in range(t)] for j in range(B)]
    den = []
    for i in range(t):
        d = 1
        for j in range(t):
            if j != i:
                d = d * (nodes[i] - nodes[j]) % p
        den.append(d)
    A = [[pow(nodes[i], s, p) for i in range(t)] for s in range(t)]
    solved = [solve_mod(A, vals[j], p) for j in range(B)]
    newton = [[divided_difference(samples, [solved[j][i] for j in range(B)], 0, d, p) for d in range(B)]
              for i in range(t)]
    return dict(p=p, anchors=anchors, samples=samples, exps=[list(e) for e in E], planted=planted,
                nodes=nodes, master=M, vals=vals, den=den, solved=solved, newton=newton)


if __name__ == "__main__":
    out = {
        "citation": "SURVEY.md 8(c).4 worked example; method: PAPER.md L19-22 (eq. 1), L55-60 (eq. 3), L191-197",
        "cases": [case(101, [2, 3], [2, 5, 7]),
                  case((1 << 63) - 25, [123456789, 987654321], [2, 3, 5])],
    }
    path = os.path.join(os.path.dirname(os.path.abspath(__file__)), "worked_example.json")
    with open(path, "w") as f:
        json.dump(out, f, indent=1)
    print("wrote", path)
