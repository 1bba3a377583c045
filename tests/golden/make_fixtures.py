"""Writes the exact-integer fixtures of this directory.  Pure Python integer arithmetic: no oracle, no
CUDA path, no floating point -- every matrix below is fixed by a textbook identity and re-verified here
by exact integer products before it is written.

  pascal8   S_ij = C(i+j, i) (symmetric Pascal matrix) = U^T U with U_ij = C(j, i) (upper Pascal matrix),
            U^-1_ij = (-1)^(i+j) C(j, i)          [e.g. Higham, Accuracy and Stability of Numerical
                                                    Algorithms, 2nd ed., section 28.4; Edelman & Strang,
                                                    "Pascal matrices", Amer. Math. Monthly 111 (2004)]
  minij12   S_ij = min(i, j) + 1 = U^T U with U = upper triangle of ones, U^-1 = I - superdiagonal
                                                   [Higham, ibid., section 28.5 (the "minij" / Lehmer family)]

H is an arbitrary symmetric integer matrix, C~ an arbitrary integer block; H~ = U^-T H U^-1 and C = U^-1 C~
are then integer matrices, computed exactly.  (PAPER.md prints no worked numerical example of steps
1-3 or of the back-transform -- its only numbers are the timings of Table 1, PAPER.md:133 -- so there is
no paper value to store; these fixtures pin the oracle to something that is neither its own output nor
a library's.)

    python tests/golden/make_fixtures.py      # rewrites pascal8.txt and minij12.txt next to this file
"""
import os
from math import comb

HERE = os.path.dirname(os.path.abspath(__file__))


def matmul(A, B):
    return [[sum(A[i][k] * B[k][j] for k in range(len(B))) for j in range(len(B[0]))] for i in range(len(A))]


def transpose(A):
    return [list(r) for r in zip(*A)]


def eye(n):
    return [[int(i == j) for j in range(n)] for i in range(n)]


def write(name, source, S, U, V):
    n = len(S)
    assert matmul(transpose(U), U) == S, "U^T U != S"
    assert matmul(U, V) == eye(n), "U V != I"
    H = [[((i + 1) * (j + 1)) % 7 - 3 + (5 if i == j else 0) for j in range(n)] for i in range(n)]
    assert H == transpose(H)
    Ht = matmul(transpose(V), matmul(H, V))
    assert Ht == transpose(Ht)
    Ct = [[((3 * i + 5 * j) % 11) - 5 for j in range(3)] for i in range(n)]
    C = matmul(V, Ct)
    with open(os.path.join(HERE, name + ".txt"), "w") as f:
        f.write(f"# {name}: {source}\n# written by tests/golden/make_fixtures.py (exact integer arithmetic); row-major rows below\n")
        f.write(f"N {n}\n")
        for key, M in (("S", S), ("U", U), ("V", V), ("H", H), ("Ht", Ht), ("Ct", Ct), ("C", C)):
            f.write(f"{key} {len(M)} {len(M[0])}\n")
            for row in M:
                f.write(" ".join(str(x) for x in row) + "\n")


def main():
    n = 8
    write("pascal8", "symmetric Pascal matrix, S_ij = C(i+j,i); U_ij = C(j,i); U^-1_ij = (-1)^(i+j) C(j,i)",
          [[comb(i + j, i) for j in range(n)] for i in range(n)],
          [[comb(j, i) for j in range(n)] for i in range(n)],
          [[(-1) ** (i + j) * comb(j, i) for j in range(n)] for i in range(n)])
    n = 12
    write("minij12", "S_ij = min(i,j)+1; U = upper triangle of ones; U^-1 = I - superdiagonal",
          [[min(i, j) + 1 for j in range(n)] for i in range(n)],
          [[int(j >= i) for j in range(n)] for i in range(n)],
          [[1 if i == j else (-1 if j == i + 1 else 0) for j in range(n)] for i in range(n)])


if __name__ == "__main__":
    main()
