"""Build-time generator of csrc/recon_gen.cuh: the constant reference-cell operators of the compact reconstruction
as fully unrolled sparse fp64 device code (one coefficient set for every cell).

  recon_Md      a = M d       34 x 72, Eq. 14/19: strict on the six face-neighbour averages, least squares on the rest
  recon_smooth  IS by derivative order of the quartic
  recon_eval    value and reference gradient of a polynomial at the 24 face Gauss points (96 x 34)

This derivation is independent of the CPU oracle (oracle/): rows come from Gauss-Legendre quadrature of the monomials
(exact for the degrees involved), the constrained least squares is solved by the null-space method.
Ordering conventions: faces m = 2*axis + (0:+,1:-); edges n = 4*z0 + 2*(s1>0) + (s2>0);
lines s = 4*axis + 2*a + b; points p = 4*m + 2*a + b; basis sorted by total degree, then d1 desc, d2 desc.
"""
import itertools
import math
import os

import numpy as np

G = 0.5 / math.sqrt(3.0)
H1, H2, H3 = 2.0, 1.0, 3.0          # h1', h2', h3'
TOL = 1e-13


def basis_indices():
    out = []
    for tot in range(1, 5):
        for d1 in range(tot, -1, -1):
            for d2 in range(tot - d1, -1, -1):
                out.append((d1, d2, tot - d1 - d2))
    return out


def other_axes(ax):
    return [a for a in range(3) if a != ax]


def face_offsets():
    out = []
    for m in range(6):
        o = [0, 0, 0]; o[m // 2] = 1 if m % 2 == 0 else -1; out.append(tuple(o))
    return out


def edge_offsets():
    out = []
    for n in range(12):
        z0 = n // 4; o1, o2 = other_axes(z0)
        o = [0, 0, 0]; o[o1] = 1 if (n >> 1) & 1 else -1; o[o2] = 1 if n & 1 else -1
        out.append((tuple(o), z0))
    return out


def gauss_points():
    pts = []
    for m in range(6):
        ax = m // 2; o1, o2 = other_axes(ax)
        for a in (0, 1):
            for b in (0, 1):
                x = [0.0, 0.0, 0.0]
                x[ax] = 0.5 if m % 2 == 0 else -0.5; x[o1] = G if a else -G; x[o2] = G if b else -G
                pts.append(x)
    return pts


_x, _w = np.polynomial.legendre.leggauss(4)      # exact to degree 7 per direction
_x = 0.5 * _x; _w = 0.5 * _w


def mono(d, x, y, z, der=None):
    """x^d0/d0! y^d1/d1! z^d2/d2!, optionally differentiated once along axis der."""
    e = list(d)
    if der is not None:
        if e[der] == 0:
            return 0.0 * x
        e[der] -= 1
    return (x ** e[0] * y ** e[1] * z ** e[2]) / (math.factorial(e[0]) * math.factorial(e[1]) * math.factorial(e[2]))


def cube_avg(d, o, der=None):
    X, Y, Z = np.meshgrid(_x + o[0], _x + o[1], _x + o[2], indexing="ij")
    W = _w[:, None, None] * _w[None, :, None] * _w[None, None, :]
    return float((W * mono(d, X, Y, Z, der)).sum())


def build_matrices():
    B = basis_indices()
    rows = []
    for d in B:
        col = []
        m0 = cube_avg(d, (0, 0, 0))
        for o in face_offsets():
            col.append(cube_avg(d, o) - m0)
        for o, _ in edge_offsets():
            col.append(cube_avg(d, o) - m0)
        for o in face_offsets():
            for ax in range(3):
                col.append(H1 * cube_avg(d, o, ax))
        for o, z0 in edge_offsets():
            col.append(H2 * cube_avg(d, o, z0))
            col.append(H2 * sum(o[ax] * cube_avg(d, o, ax) for ax in range(3)) / math.sqrt(2.0))
        for ax in range(3):
            o1, o2 = other_axes(ax)
            for a in (0, 1):
                for b in (0, 1):
                    x1 = [0.0, 0.0, 0.0]; x2 = [0.0, 0.0, 0.0]
                    x1[ax] = -0.5; x2[ax] = 0.5
                    x1[o1] = x2[o1] = G if a else -G; x1[o2] = x2[o2] = G if b else -G
                    one = np.array(1.0)
                    col.append(H3 * float(mono(d, one * x2[0], one * x2[1], one * x2[2]) - mono(d, one * x1[0], one * x1[1], one * x1[2])))
        rows.append(col)
    A = np.array(rows).T                      # 72 x 34
    C, L = A[:6], A[6:]
    # null-space method: a = C^+ c + Z y,  y = argmin |L Z y - (l - L C^+ c)|
    Cp = np.linalg.pinv(C)
    _, _, Vt = np.linalg.svd(C)
    Z = Vt[6:].T
    LZp = np.linalg.pinv(L @ Z)
    M = np.zeros((34, 72))
    M[:, :6] = Cp - Z @ LZp @ L @ Cp
    M[:, 6:] = Z @ LZp
    # evaluation matrix
    E = np.zeros((96, 34))
    one = np.array(1.0)
    for p, x in enumerate(gauss_points()):
        for b, d in enumerate(B):
            E[4 * p, b] = float(mono(d, one * x[0], one * x[1], one * x[2])) - cube_avg(d, (0, 0, 0))
            for ax in range(3):
                E[4 * p + 1 + ax, b] = float(mono(d, one * x[0], one * x[1], one * x[2], ax))
    # Gram matrices of the smoothness indicators per derivative order
    X, Y, Zz = np.meshgrid(_x, _x, _x, indexing="ij")
    W = _w[:, None, None] * _w[None, :, None] * _w[None, None, :]
    Gram = np.zeros((4, 34, 34))
    for l in itertools.product(range(5), repeat=3):
        o = sum(l)
        if not 1 <= o <= 4:
            continue
        ders = []
        for d in B:
            e = [d[i] - l[i] for i in range(3)]
            ders.append(None if min(e) < 0 else mono(e, X, Y, Zz))
        for i in range(34):
            if ders[i] is None:
                continue
            for j in range(34):
                if ders[j] is None:
                    continue
                Gram[o - 1, i, j] += float((W * ders[i] * ders[j]).sum())
    return M, E, Gram


def lit(v):
    return repr(float(v))


def emit_linear(name, Mx, nin, nout, xin, xout):
    lines = ["__device__ __forceinline__ void %s(const double* __restrict__ %s, double* __restrict__ %s) {" % (name, xin, xout)]
    for i in range(nout):
        terms = ["%s * %s[%d]" % (lit(Mx[i, c]), xin, c) for c in range(nin) if abs(Mx[i, c]) > TOL]
        lines.append("  %s[%d] = %s;" % (xout, i, " + ".join(terms) if terms else "0.0"))
    lines.append("}")
    return "\n".join(lines)


def emit_quadform(name, Gm):
    """s = sum_i a_i (G_ii a_i + 2 sum_{j>i} G_ij a_j)"""
    parts = []
    for i in range(34):
        inner = []
        if abs(Gm[i, i]) > TOL:
            inner.append("%s * a[%d]" % (lit(Gm[i, i]), i))
        for j in range(i + 1, 34):
            if abs(Gm[i, j]) > TOL:
                inner.append("%s * a[%d]" % (lit(2.0 * Gm[i, j]), j))
        if inner:
            parts.append("a[%d] * (%s)" % (i, " + ".join(inner)))
    return "__device__ __forceinline__ double %s(const double* __restrict__ a) {\n  return %s;\n}" % (name, "\n       + ".join(parts))


def generate(path):
    M, E, Gram = build_matrices()
    nnzM = int((np.abs(M) > TOL).sum()); nnzE = int((np.abs(E) > TOL).sum())
    out = ["// GENERATED by gen_recon.py -- do not edit.  M: %d non-zeros of %d, E: %d of %d." % (nnzM, M.size, nnzE, E.size),
           "#pragma once",
           "#define CGKS_NNZ_M %d" % nnzM, "#define CGKS_NNZ_E %d" % nnzE,
           emit_linear("recon_Md", M, 72, 34, "d", "a"),
           emit_quadform("recon_IS1", Gram[0]),
           emit_quadform("recon_IS2", Gram[1]),
           emit_quadform("recon_IS34", Gram[2] + Gram[3]),
           emit_linear("recon_eval", E, 34, 96, "c", "o"), ""]
    with open(path, "w") as f:
        f.write("\n".join(out))
    return M, E, Gram


if __name__ == "__main__":
    here = os.path.dirname(os.path.abspath(__file__))
    M, E, Gram = generate(os.path.join(here, "recon_gen.cuh"))
    print("wrote recon_gen.cuh: nnz M", int((np.abs(M) > TOL).sum()), "nnz E", int((np.abs(E) > TOL).sum()))
