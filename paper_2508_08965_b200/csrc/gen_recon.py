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
    return M, E, Gram, A


CANON = []      # canonical values of the emitted constants


def lit(v):
    """A coefficient as a literal.  Coefficients that are mathematically equal come out of the numerical null-space / quadrature
    construction with different last bits; they are snapped to one representative (relative distance <= 1e-13), so that
    ptxas can share the two UMOV instructions that materialise an FP64 literal among the FMAs that use it."""
    v = float(v)
    for c in CANON:
        if abs(v - c) <= 1e-13 * abs(c):
            return repr(c)
        if abs(v + c) <= 1e-13 * abs(c):
            return repr(-c)
    CANON.append(v)
    return repr(v)


# ------------------------------------------------------------------------------------------------------------------
# Symmetry reduction.  The reference stencil, the data functionals of Eq. 19 and the 24 face Gauss points are invariant
# under the three reflections xi_ax -> -xi_ax, so M and E commute with them: in a basis of reflection-parity
# combinations of the data (sums/differences over each orbit) M is block diagonal over the 8 parity classes of the
# monomials (330 non-zeros instead of 1008), and the 8 Gauss points of a face pair are one orbit: their values follow
# from 8 class sums at ONE representative point by a three-stage add/subtract butterfly.
def data_groups():
    """Neighbour groups of the 72 data: (name, [global d indices in local order], [scale of each: d = scale * raw])."""
    groups = []
    for ax in range(3):          # face pair: x[0] = dq(+), x[1] = dq(-), x[2..4] = gr'(+), x[5..7] = gr'(-)
        mp, mm = 2 * ax, 2 * ax + 1
        idx = [mp, mm] + [18 + 3 * mp + a for a in range(3)] + [18 + 3 * mm + a for a in range(3)]
        groups.append(("face%d" % ax, idx, [1.0, 1.0] + [H1] * 6))
    for z0 in range(3):          # edge quad t = 0..3: x[t] = dq, x[4+2t] = gr'[z0], x[5+2t] = o.gr' (no 1/sqrt 2)
        idx = [6 + 4 * z0 + t for t in range(4)]
        sc = [1.0] * 4
        for t in range(4):
            e = 4 * z0 + t
            idx += [36 + 2 * e, 37 + 2 * e]; sc += [H2, H2 / math.sqrt(2.0)]
        groups.append(("edge%d" % z0, idx, sc))
    for ax in range(3):          # lines along ax: x[t] = D[4 ax + t] (no factor h3')
        groups.append(("line%d" % ax, [60 + 4 * ax + t for t in range(4)], [H3] * 4))
    return groups


def reflections(A, B):
    """Signed permutations of the data functionals: f_i(p o R_ax) = sg[i] * f_perm[i](p)."""
    out = []
    for ax in range(3):
        AS = A * np.array([(-1.0) ** d[ax] for d in B])[None, :]
        perm = np.zeros(72, int); sg = np.zeros(72)
        for i in range(72):
            hit = [(j, s) for j in range(72) for s in (1.0, -1.0) if np.allclose(AS[i], s * A[j], atol=1e-11)]
            assert len(hit) == 1, (ax, i, hit)
            perm[i], sg[i] = hit[0]
        R = np.zeros((72, 72))
        R[np.arange(72), perm] = sg
        out.append(R)
    return out


def parity_combos(A, B, M):
    """For every group: list of orbits; per orbit (members [global idx], rows t (+-1, shape s x s), columns of M')."""
    R = reflections(A, B)
    bcls = [tuple(d[i] % 2 for i in range(3)) for d in B]
    groups = data_groups()
    scale = np.zeros(72)
    for _, idx, sc in groups:
        scale[idx] = sc
    res = []
    nnz = 0
    for name, idx, sc in groups:
        left = list(idx); orbits = []
        while left:
            i0 = left[0]
            imgs = set()
            for pw in itertools.product((0, 1), repeat=3):          # images of datum i0 under the 8 reflections
                v = np.eye(72)[i0]
                for ax in range(3):
                    if pw[ax]:
                        v = v @ R[ax]
                imgs.add(int(np.nonzero(v)[0][0]))
            members = sorted(imgs, key=idx.index)
            assert all(m in left for m in members)
            for m in members:
                left.remove(m)
            s_ = len(members)
            assert s_ in (2, 4)
            rows = []; cols = []
            for c in itertools.product((0, 1), repeat=3):
                P = np.eye(72)
                for ax in range(3):
                    P = P @ (np.eye(72) + (-1.0) ** c[ax] * R[ax]) / 2.0
                r = P[members[0]]
                if np.abs(r).max() < 1e-12:
                    continue
                assert np.abs(np.delete(r, members)).max() < 1e-12
                t = np.sign(r[members])
                assert np.all(np.abs(t) == 1.0)
                full = np.zeros(72); full[members] = t
                assert abs(scale[members].max() - scale[members].min()) < 1e-15
                col = M @ full * scale[members[0]] / s_
                nzb = [b for b in range(34) if abs(col[b]) > TOL]
                assert all(bcls[b] == c for b in nzb), (name, c)
                rows.append(t); cols.append(col); nnz += len(nzb)
            assert len(rows) == s_
            orbits.append(([idx.index(m) for m in members], np.array(rows), cols))
        res.append((name, len(idx), orbits))
    return res, nnz


def emit_group(name, nloc, orbits):
    """a[] += M' * (parity combinations of this group's raw data x[0..nloc-1])."""
    L = ["__device__ __forceinline__ void recon_acc_%s(const double* __restrict__ x, double* __restrict__ a) {" % name]
    uid = 0
    for members, T, cols in orbits:
        s_ = len(members)
        Tn = T * T[0][None, :]                 # column signs of row 0 folded into y
        y = []
        for q, m in enumerate(members):
            y.append("x[%d]" % m if T[0][q] > 0 else "(-x[%d])" % m)
        combos = [None] * s_
        pre = "%s_%d" % (name, uid); uid += 1
        if s_ == 2:
            L.append("  const double %s_p = %s + %s, %s_m = %s - %s;" % (pre, y[0], y[1], pre, y[0], y[1]))
            for r in range(2):
                combos[r] = "%s_p" % pre if Tn[r][1] > 0 else "%s_m" % pre
        else:
            r1 = 1
            plus = [q for q in range(4) if Tn[r1][q] > 0]; minus = [q for q in range(4) if Tn[r1][q] < 0]
            assert len(plus) == 2 and len(minus) == 2 and 0 in plus
            p_, q_ = plus; r_, s2 = minus
            L.append("  const double %s_up = %s + %s, %s_um = %s - %s, %s_vp = %s + %s, %s_vm = %s - %s;"
                     % (pre, y[p_], y[q_], pre, y[p_], y[q_], pre, y[r_], y[s2], pre, y[r_], y[s2]))
            for r in range(4):
                row = Tn[r]
                if row[p_] == row[q_]:         # symmetric within the pairs
                    assert row[r_] == row[s2]
                    sgn = "+" if row[r_] * row[p_] > 0 else "-"
                    e = "%s_up %s %s_vp" % (pre, sgn, pre)
                    if row[p_] < 0:
                        e = "-(%s)" % e
                else:
                    assert row[r_] != row[s2]
                    sgn = "+" if row[r_] * row[p_] > 0 else "-"
                    e = "%s_um %s %s_vm" % (pre, sgn, pre)
                    if row[p_] < 0:
                        e = "-(%s)" % e
                L.append("  const double %s_c%d = %s;" % (pre, r, e))
                combos[r] = "%s_c%d" % (pre, r)
        for r in range(s_):
            for b in range(34):
                if abs(cols[r][b]) > TOL:
                    L.append("  a[%d] = fma(%s, %s, a[%d]);" % (b, lit(cols[r][b]), combos[r], b))
    L.append("}")
    return "\n".join(L)


def emit_eval_axis(ax, B, volume=False):
    """Value and reference gradient at the 8 Gauss points of the face pair of axis ax: out[4*(4*sgn + 2*a + b) + kappa],
    sgn = 0 for the + face; (a, b) select -g/+g on the two other axes (ascending); kappa = 0 value, 1..3 d/dxi_r.
    volume=True: the 8 interior Gauss points (+-g, +-g, +-g) of the 2x2x2 rule instead (ax = 0; sgn = 0 selects +g)."""
    o1, o2 = other_axes(ax)
    xs = [0.0, 0.0, 0.0]; xs[ax] = G if volume else 0.5; xs[o1] = G; xs[o2] = G
    one = np.array(1.0)
    L = ["__device__ __forceinline__ void recon_eval_%s(const double* __restrict__ a, double* __restrict__ out) {"
         % ("volume" if volume else "axis%d" % ax)]
    for kap in range(4):
        sums = {}
        for b, d in enumerate(B):
            if kap == 0:
                cf = float(mono(d, one * xs[0], one * xs[1], one * xs[2])) - cube_avg(d, (0, 0, 0)); e = list(d)
            else:
                if d[kap - 1] == 0:
                    continue
                cf = float(mono(d, one * xs[0], one * xs[1], one * xs[2], kap - 1)); e = list(d); e[kap - 1] -= 1
            if abs(cf) < TOL:
                continue
            c = (e[ax] % 2, e[o1] % 2, e[o2] % 2)
            sums.setdefault(c, []).append((b, cf))
        V = {}
        for c, terms in sorted(sums.items()):
            nm = "v%d_%d%d%d" % (kap, c[0], c[1], c[2])
            expr = "%s * a[%d]" % (lit(terms[0][1]), terms[0][0])
            for b, cf in terms[1:]:
                expr = "fma(%s, a[%d], %s)" % (lit(cf), b, expr)
            L.append("  const double %s = %s;" % (nm, expr))
            V[c] = nm
        # three butterfly stages: class bit -> sign of the coordinate
        for stage in range(3):
            Vn = {}
            for key in itertools.product((0, 1), repeat=3):
                if key[stage] == 1:
                    continue
                k0 = key; k1 = tuple(1 if i == stage else key[i] for i in range(3))
                e0, e1 = V.get(k0), V.get(k1)
                for sg in (0, 1):          # 0: coordinate positive, 1: negative
                    kk = tuple(sg if i == stage else key[i] for i in range(3))
                    nm = "w%d_%d_%d%d%d" % (kap, stage, kk[0], kk[1], kk[2])
                    if e0 is None and e1 is None:
                        continue
                    if e1 is None:
                        Vn[kk] = e0; continue
                    if e0 is None:
                        L.append("  const double %s = %s%s;" % (nm, "" if sg == 0 else "-", e1)); Vn[kk] = nm; continue
                    L.append("  const double %s = %s %s %s;" % (nm, e0, "+" if sg == 0 else "-", e1)); Vn[kk] = nm
            V = Vn
        for sgn in (0, 1):
            for a_ in (0, 1):
                for b_ in (0, 1):
                    key = (sgn, 1 - a_, 1 - b_)       # a = 1 selects +g (coordinate positive -> key bit 0)
                    L.append("  out[%d] = %s;" % (4 * (4 * sgn + 2 * a_ + b_) + kap, V.get(key, "0.0")))
    L.append("}")
    return "\n".join(L)


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
    del CANON[:]
    M, E, Gram, A = build_matrices()
    B = basis_indices()
    combos, nnzS = parity_combos(A, B, M)
    nnzM = int((np.abs(M) > TOL).sum()); nnzE = int((np.abs(E) > TOL).sum())
    out = ["// GENERATED by gen_recon.py -- do not edit.  M: %d non-zeros of %d (%d after the reflection-parity reduction), "
           "E: %d of %d." % (nnzM, M.size, nnzS, nnzE, E.size),
           "#pragma once",
           "#define CGKS_NNZ_M %d" % nnzM, "#define CGKS_NNZ_MSYM %d" % nnzS, "#define CGKS_NNZ_E %d" % nnzE]
    for name, nloc, orbits in combos:
        out.append(emit_group(name, nloc, orbits))
    out += [emit_quadform("recon_IS1", Gram[0]), emit_quadform("recon_IS2", Gram[1]),
            emit_quadform("recon_IS34", Gram[2] + Gram[3])]
    for ax in range(3):
        out.append(emit_eval_axis(ax, B))
    out.append(emit_eval_axis(0, B, volume=True))
    out.append("")
    with open(path, "w") as f:
        f.write("\n".join(out))
    return M, E, Gram, A, combos


def self_check():
    """The symmetry-reduced operators reproduce a = M d and o = E a (numpy emulation of the emitted structure)."""
    M, E, Gram, A = build_matrices()
    B = basis_indices()
    combos, nnz = parity_combos(A, B, M)
    rng = np.random.default_rng(0)
    d = rng.standard_normal(72)
    groups = data_groups()
    a = np.zeros(34)
    for (name, idx, sc), (_, nloc, orbits) in zip(groups, combos):
        raw = d[idx] / np.array(sc)
        for members, T, cols in orbits:
            for r in range(len(members)):
                a += np.array(cols[r]) * float(T[r] @ raw[members])
    assert np.abs(a - M @ d).max() < 1e-12, np.abs(a - M @ d).max()
    return nnz


if __name__ == "__main__":
    here = os.path.dirname(os.path.abspath(__file__))
    nnz = self_check()
    M, E, Gram, A, combos = generate(os.path.join(here, "recon_gen.cuh"))
    print("wrote recon_gen.cuh: nnz M", int((np.abs(M) > TOL).sum()), "-> symmetric", nnz, "; nnz E", int((np.abs(E) > TOL).sum()))
