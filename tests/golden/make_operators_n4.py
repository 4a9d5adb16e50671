"""Writes tests/golden/operators_n4.txt: the n = 4 operators Upsilon (4x4) and Xi (4x2), derived
EXACTLY (SymPy, radicals) from the definitions Eq. 11-13 of PAPER.md (M, A, Gamma as integrals of
Lagrange polynomials through the roots of (1-x^2)P_3'(x); Upsilon = M^-1 A^T-type product, Xi =
M^-1 Gamma) -- not from the closed forms Eq. 54/57 that oracle/basis.py restates.  Calls neither
oracle/ nor the CUDA path.   Usage: python tests/golden/make_operators_n4.py"""
import os
import sympy as sp

x = sp.symbols("x")
n = 4
P3 = sp.legendre(3, x)
nodes = sorted(sp.solve(sp.expand((1 - x ** 2) * sp.diff(P3, x)), x), key=lambda r: float(r))
ell = []
for j in range(n):
    e = sp.Integer(1)
    for k in range(n):
        if k != j:
            e *= (x - nodes[k]) / (nodes[j] - nodes[k])
    ell.append(sp.expand(e))
M = sp.Matrix(n, n, lambda i, j: sp.integrate(ell[i] * ell[j], (x, -1, 1)))
# weak form Eq. 9: du_b/dt <l_b|l_g> = F_b <l_b | d l_g> - Flux_b <l_b|l_g>_boundary
Adv = sp.Matrix(n, n, lambda b, g: sp.integrate(ell[b] * sp.diff(ell[g], x), (x, -1, 1)))   # <l_b | l_g'>
Minv = M.inv()
Ups = sp.simplify(Minv * Adv.T)          # Ups[g, b]: (Ups F)_g = sum_b Ups[g,b] F_b
Xi = sp.simplify(Minv[:, [0, n - 1]])    # face mass = delta at the end nodes
out = os.path.join(os.path.dirname(os.path.abspath(__file__)), "operators_n4.txt")
with open(out, "w") as fh:
    fh.write("# n = 4 LGL operators, exact from Eq. 11-13 of PAPER.md (arXiv 2202.13532), by make_operators_n4.py\n")
    fh.write("# rows 1-4: Upsilon[j][k] (row = output node j); rows 5-8: Xi[j][L,R]\n")
    for i in range(n):
        fh.write(" ".join(sp.N(Ups[i, j], 20).__str__() for j in range(n)) + "\n")
    for i in range(n):
        fh.write(" ".join(sp.N(Xi[i, j], 20).__str__() for j in range(2)) + "\n")
print(open(out).read())
