"""Test helper: builds the 72-entry data vector of Eq. 14/19 for an arbitrary smooth
field on the reference lattice by NUMERICAL quadrature, independently of the oracle's closed-form row integrals.

Ordering conventions are the ones documented in DESIGN.md section 2 (faces m = 2*axis + (0:+, 1:-); edges
n = 4*z0 + 2*(s1>0) + (s2>0); lines s = 4*axis + 2*a + b)."""
import itertools
import math

import numpy as np

G = 0.5 / math.sqrt(3.0)
_gl_x, _gl_w = np.polynomial.legendre.leggauss(8)
_gl_x = 0.5 * _gl_x; _gl_w = 0.5 * _gl_w          # rule on [-1/2, 1/2]


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


def cube_avg(fn, o):
    """Average of fn(x,y,z) over the unit cube centred at integer offset o (tensor Gauss-Legendre)."""
    X, Y, Z = np.meshgrid(_gl_x + o[0], _gl_x + o[1], _gl_x + o[2], indexing="ij")
    W = _gl_w[:, None, None] * _gl_w[None, :, None] * _gl_w[None, None, :]
    return float((W * fn(X, Y, Z)).sum())


def line_points():
    """[(x1, x2)] for the 12 lines."""
    out = []
    for ax in range(3):
        o1, o2 = other_axes(ax)
        for a in (0, 1):
            for b in (0, 1):
                x1 = [0.0, 0.0, 0.0]; x2 = [0.0, 0.0, 0.0]
                x1[ax] = -0.5; x2[ax] = 0.5
                x1[o1] = x2[o1] = G if a else -G
                x1[o2] = x2[o2] = G if b else -G
                out.append((x1, x2))
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
    return np.array(pts)


def data_vector(fn, grad):
    """fn(x,y,z) -> value; grad(x,y,z) -> tuple of the three partial derivatives.  Returns (q0, d[72])."""
    q0 = cube_avg(fn, (0, 0, 0))
    d = []
    for o in face_offsets():
        d.append(cube_avg(fn, o) - q0)
    for o, _ in edge_offsets():
        d.append(cube_avg(fn, o) - q0)
    for o in face_offsets():
        for ax in range(3):
            d.append(2.0 * cube_avg(lambda x, y, z: grad(x, y, z)[ax], o))
    for o, z0 in edge_offsets():
        gr = [cube_avg(lambda x, y, z: grad(x, y, z)[ax], o) for ax in range(3)]
        d.append(1.0 * gr[z0])
        d.append(1.0 * sum(o[ax] * gr[ax] for ax in range(3)) / math.sqrt(2.0))
    for x1, x2 in line_points():
        d.append(3.0 * (float(fn(*x2)) - float(fn(*x1))))
    return q0, np.array(d)


def quartic_multi_indices():
    return [d for d in itertools.product(range(5), repeat=3) if sum(d) <= 4]


def poly_fn(coef):
    """coef: dict multi-index -> coefficient of x^d0 y^d1 z^d2 (plain monomials)."""
    def fn(x, y, z):
        return sum(c * x ** d[0] * y ** d[1] * z ** d[2] for d, c in coef.items())

    def grad(x, y, z):
        gx = sum(c * d[0] * x ** (d[0] - 1) * y ** d[1] * z ** d[2] for d, c in coef.items() if d[0] > 0)
        gy = sum(c * d[1] * x ** d[0] * y ** (d[1] - 1) * z ** d[2] for d, c in coef.items() if d[1] > 0)
        gz = sum(c * d[2] * x ** d[0] * y ** d[1] * z ** (d[2] - 1) for d, c in coef.items() if d[2] > 0)
        return (gx + 0 * x, gy + 0 * x, gz + 0 * x)
    return fn, grad
