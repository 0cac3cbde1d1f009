"""Pins for the oracle's local tricubic interpolation.

Nothing here retypes the oracle's formula: the references are node identities, polynomial
exactness, continuity, and scipy's barycentric interpolator.
"""
import itertools
import math

import numpy as np
import pytest
from scipy.interpolate import BarycentricInterpolator

from paper_2604_07617_b200 import workloads as W


def _grid_nodes(lo, hi, ncell):
    return [lo[d] + (hi[d] - lo[d]) * np.arange(3 * ncell[d] + 1) / (3.0 * ncell[d]) for d in range(3)]


def _field(O, coord, ncell, lo, hi, funcs, nfp=1):
    X = np.meshgrid(*_grid_nodes(lo, hi, ncell), indexing="ij")
    nodes = np.stack([fn(*X) for fn in funcs])
    fd = dict(coord=coord, ncell=ncell, lo=lo, hi=hi, nfp=nfp, nquant=len(funcs), nodes=nodes,
              G0=1.0, I0=0.0, iota0=0.4, iota1=0.0, psi0=1.0)
    return O.Field(fd), nodes


def test_lagrange_cardinal_and_partition_of_unity(oracle):
    O = oracle
    for j in range(4):
        L = O.lagrange4(j / 3.0)
        want = np.zeros(4)
        want[j] = 1.0
        assert np.allclose(L, want, atol=2e-16)
    for u in np.linspace(-0.7, 1.9, 41):
        L = O.lagrange4(float(u))
        assert abs(L.sum() - 1.0) < 1e-13
        # first moment: sum_a L_a(u) * (a/3) = u  (a dropped/permuted basis function breaks it)
        assert abs((L * np.arange(4) / 3.0).sum() - u) < 1e-13


def test_matches_scipy_barycentric_1d(oracle):
    O = oracle
    rng = np.random.default_rng(5)
    f = rng.normal(size=4)
    ref = BarycentricInterpolator(np.arange(4) / 3.0, f)
    for u in rng.uniform(-0.5, 1.5, size=20):
        assert abs(O.lagrange4(float(u)) @ f - float(ref(u))) < 1e-13 * (1 + abs(float(ref(u))))


@pytest.mark.parametrize("coord", [0, 1])
def test_node_values_reproduced_exactly(oracle, coord):
    O = oracle
    rng = np.random.default_rng(11)
    ncell = [3, 2, 4]
    lo = [0.0, 0.0, 0.0] if coord == 0 else [1.0, -2.0, 0.0]
    hi = [1.0, 2 * math.pi, 2 * math.pi / 4] if coord == 0 else [3.0, 2.0, 2 * math.pi]
    n = [3 * k + 1 for k in ncell]
    nodes = rng.normal(size=(2, *n))
    fd = dict(coord=coord, ncell=ncell, lo=lo, hi=hi, nfp=4 if coord == 0 else 1, nquant=2,
              nodes=nodes, G0=1.0, I0=0.0, iota0=0.4, iota1=0.0, psi0=1.0)
    f = O.Field(fd)
    g = _grid_nodes(lo, hi, ncell)
    periodic = [False, True, True] if coord == 0 else [False, False, True]
    for _ in range(200):
        j = [int(rng.integers(0, n[d])) for d in range(3)]
        x = [g[d][j[d]] for d in range(3)]
        got = O.tricubic(f, x)
        jj = [0 if (periodic[d] and j[d] == n[d] - 1) else j[d] for d in range(3)]
        # a periodic end node is looked up as the first node; the generator duplicates it, random
        # data here does not, so compare against the node the reduction lands on
        want = nodes[:, jj[0], jj[1], jj[2]]
        assert np.allclose(got, want, rtol=0, atol=1e-13 * np.abs(nodes).max())


@pytest.mark.parametrize("coord", [0, 1])
def test_tricubic_polynomial_reproduced_including_extrapolation(oracle, coord):
    O = oracle
    rng = np.random.default_rng(7)
    coef = rng.normal(size=(4, 4, 4))

    def P(x, y, z):
        out = 0.0
        for i, j, k in itertools.product(range(4), repeat=3):
            out = out + coef[i, j, k] * x ** i * y ** j * z ** k
        return out

    ncell = [3, 2, 4]
    lo = [0.0, 0.0, 0.0] if coord == 0 else [1.0, -2.0, 0.0]
    hi = [1.0, 2 * math.pi, 2 * math.pi / 4] if coord == 0 else [3.0, 2.0, 2 * math.pi]
    f, _ = _field(O, coord, ncell, lo, hi, [P, lambda x, y, z: 2.0 - P(x, y, z)], nfp=4 if coord == 0 else 1)
    pts = []
    for _ in range(100):
        x = [lo[d] + (hi[d] - lo[d]) * rng.random() for d in range(3)]
        pts.append(x)
    # extrapolation in the non-periodic dims
    for _ in range(50):
        x = [lo[d] + (hi[d] - lo[d]) * rng.random() for d in range(3)]
        x[0] = hi[0] + 0.3 * (hi[0] - lo[0]) * rng.random() if rng.random() < 0.5 else lo[0] - 0.2 * rng.random()
        if coord == 1:
            x[1] = hi[1] + 0.5 * rng.random()
        pts.append(x)
    for x in pts:
        got = O.tricubic(f, x)
        want = P(*x)
        scale = sum(abs(coef[i, j, k]) * abs(x[0]) ** i * abs(x[1]) ** j * abs(x[2]) ** k
                    for i, j, k in itertools.product(range(4), repeat=3))
        assert abs(got[0] - want) <= 1e-13 * scale * 20
        assert abs(got[1] - (2.0 - want)) <= 1e-13 * scale * 20


def test_axes_not_transposed(oracle):
    """f = x0 + 10 x1 + 100 x2 is degree 1 per variable: any swapped axis or basis vector shows."""
    O = oracle
    f, _ = _field(O, 1, [2, 3, 4], [1.0, -2.0, 0.0], [3.0, 2.0, 2 * math.pi],
                  [lambda x, y, z: x + 10 * y + 100 * z])
    rng = np.random.default_rng(3)
    for _ in range(50):
        x = [1 + 2 * rng.random(), -2 + 4 * rng.random(), 2 * math.pi * rng.random()]
        assert abs(O.tricubic(f, x)[0] - (x[0] + 10 * x[1] + 100 * x[2])) < 1e-11


def test_continuity_across_cell_faces(oracle):
    O = oracle
    rng = np.random.default_rng(13)
    ncell = [3, 3, 3]
    lo, hi = [0.0, 0.0, 0.0], [1.0, 2 * math.pi, 2 * math.pi / 4]
    g = lambda s, t, z: np.cos(3 * s) * np.sin(t + 0.3) * np.cos(4 * z) + s * s
    f, _ = _field(O, 0, ncell, lo, hi, [g], nfp=4)
    for d in range(3):
        h = (hi[d] - lo[d]) / ncell[d]
        for face in range(1, ncell[d]):
            for _ in range(10):
                x = [lo[e] + (hi[e] - lo[e]) * rng.random() for e in range(3)]
                xm, xp = list(x), list(x)
                xm[d] = lo[d] + face * h - 1e-13
                xp[d] = lo[d] + face * h + 1e-13
                cm, _ = O.locate(f, xm)
                cp, _ = O.locate(f, xp)
                assert cp[d] == cm[d] + 1
                assert abs(O.tricubic(f, xm)[0] - O.tricubic(f, xp)[0]) < 1e-11


def test_successive_1d_barycentric(oracle):
    """Special case that reduces to a library routine: three successive 1-D interpolations."""
    O = oracle
    rng = np.random.default_rng(17)
    ncell = [2, 2, 2]
    lo, hi = [0.0, 0.0, 0.0], [1.0, 2 * math.pi, 2 * math.pi]
    n = [7, 7, 7]
    nodes = rng.normal(size=(1, *n))
    fd = dict(coord=0, ncell=ncell, lo=lo, hi=hi, nfp=1, nquant=1, nodes=nodes, G0=1.0, I0=0.0,
              iota0=0.4, iota1=0.0, psi0=1.0)
    f = O.Field(fd)
    g = _grid_nodes(lo, hi, ncell)
    for _ in range(40):
        x = [lo[d] + (hi[d] - lo[d]) * rng.random() for d in range(3)]
        c = [min(int((x[d] - lo[d]) / ((hi[d] - lo[d]) / 2)), 1) for d in range(3)]
        blk = nodes[0, 3 * c[0]:3 * c[0] + 4, 3 * c[1]:3 * c[1] + 4, 3 * c[2]:3 * c[2] + 4]
        v2 = BarycentricInterpolator(g[2][3 * c[2]:3 * c[2] + 4], np.moveaxis(blk, 2, 0))(x[2])
        v1 = BarycentricInterpolator(g[1][3 * c[1]:3 * c[1] + 4], np.moveaxis(v2, 1, 0))(x[1])
        v0 = BarycentricInterpolator(g[0][3 * c[0]:3 * c[0] + 4], v1)(x[0])
        assert abs(O.tricubic(f, x)[0] - float(v0)) < 1e-12


def test_locate_edges_and_periodic_wrap(oracle):
    O = oracle
    f, _ = _field(O, 0, [4, 5, 6], [0.0, 0.0, 0.0], [1.0, 2 * math.pi, 2 * math.pi / 4],
                  [lambda s, t, z: s + 0 * t + 0 * z], nfp=4)
    cell, u = O.locate(f, [1.0, 0.0, 0.0])          # upper edge: last cell, u = 1 (reading Q8)
    assert cell[0] == 3 and abs(u[0] - 1.0) < 1e-15
    cell, u = O.locate(f, [1.3, 0.0, 0.0])          # beyond: nearest cell, u > 1
    assert cell[0] == 3 and abs(u[0] - (1.3 * 4 - 3)) < 1e-14
    cell, u = O.locate(f, [-0.1, 0.0, 0.0])
    assert cell[0] == 0 and abs(u[0] + 0.4) < 1e-14
    cell, u = O.locate(f, [0.5, -0.1, 2 * math.pi / 4 + 0.01])  # periodic wrap
    h1 = 2 * math.pi / 5
    assert cell[1] == 4 and abs(u[1] - ((2 * math.pi - 0.1) / h1 - 4)) < 1e-12
    assert cell[2] == 0 and abs(u[2] - 0.01 / (2 * math.pi / 4 / 6)) < 1e-12
    cell, u = O.locate(f, [0.5, 2 * math.pi, 0.0])
    assert cell[1] == 0 and abs(u[1]) < 1e-15
    # s and the periodic theta after many turns
    cell, u = O.locate(f, [0.5, 0.3 + 40 * math.pi, 0.0])
    assert cell[1] == 0 and abs(u[1] - 0.3 / h1) < 1e-10


def test_field_build_bruteforce_and_size(oracle):
    """64 k^3 rows x m columns, rows of a cell contiguous, faces duplicated."""
    O = oracle
    rng = np.random.default_rng(19)
    ncell = [2, 3, 2]
    n = [3 * k + 1 for k in ncell]
    nodes = rng.normal(size=(3, *n))
    fd = dict(coord=0, ncell=ncell, lo=[0, 0, 0], hi=[1, 1, 1], nfp=1, nquant=3, nodes=nodes,
              G0=1.0, I0=0.0, iota0=0.4, iota1=0.0, psi0=1.0)
    f = O.Field(fd)
    tab = O.field_build(f)
    assert tab.shape == (64 * 2 * 3 * 2, 3)
    for _ in range(500):
        i = [int(rng.integers(0, ncell[d])) for d in range(3)]
        a = [int(rng.integers(0, 4)) for _ in range(3)]
        q = int(rng.integers(0, 3))
        cell = (i[0] * ncell[1] + i[1]) * ncell[2] + i[2]
        node = (a[0] * 4 + a[1]) * 4 + a[2]
        assert tab[cell * 64 + node, q] == nodes[q, 3 * i[0] + a[0], 3 * i[1] + a[1], 3 * i[2] + a[2]]
    # shared face stored twice with identical values: node a0=3 of cell i0 == node a0=0 of cell i0+1
    c0 = (0 * 3 + 1) * 2 + 1
    c1 = (1 * 3 + 1) * 2 + 1
    for b in range(4):
        for c in range(4):
            assert np.array_equal(tab[c0 * 64 + (3 * 4 + b) * 4 + c], tab[c1 * 64 + (0 * 4 + b) * 4 + c])


# ---- reading R1c: the gradient of the interpolant (derivative-of-interpolant mode) ---------------
def test_gradient_of_the_interpolant_is_exact_for_tricubics(oracle):
    """The local tricubic reproduces any polynomial of degree <= 3 per variable; so does its gradient, inside the
    grid and where the end cells are extrapolated."""
    O = oracle
    rng = np.random.default_rng(5)
    c = rng.normal(size=(4, 4, 4))
    lo, hi, k = [0.0, -1.0, 2.0], [1.0, 1.0, 3.5], [2, 3, 2]
    ax = [np.linspace(lo[d], hi[d], 3 * k[d] + 1) for d in range(3)]
    P = lambda x, y, z: sum(c[i, j, l] * x ** i * y ** j * z ** l for i in range(4) for j in range(4) for l in range(4))
    dP = lambda x, y, z: np.array([
        sum(i * c[i, j, l] * x ** (i - 1) * y ** j * z ** l for i in range(1, 4) for j in range(4) for l in range(4)),
        sum(j * c[i, j, l] * x ** i * y ** (j - 1) * z ** l for i in range(4) for j in range(1, 4) for l in range(4)),
        sum(l * c[i, j, l] * x ** i * y ** j * z ** (l - 1) for i in range(4) for j in range(4) for l in range(1, 4))])
    X, Y, Z = np.meshgrid(*ax, indexing="ij")
    fd = dict(coord=1, ncell=k, lo=lo, hi=hi, nfp=1, nquant=1, nodes=P(X, Y, Z)[None], G0=1.0, I0=0.0, iota0=0.0,
              iota1=0.0, psi0=1.0)        # cylindrical grid: only the last dimension is periodic
    f = O.Field(fd)
    for x in ([0.3, 0.1, 2.2], [0.77, -0.93, 3.4], [1.08, 1.05, 2.9], [-0.04, 0.5, 2.01]):
        v, g = O.tricubic_grad(f, x)
        assert abs(v - P(*x)) <= 1e-12 * (1 + abs(P(*x)))
        assert np.all(np.abs(g - dP(*x)) <= 1e-11 * (1 + np.abs(dP(*x))))


def test_gradient_of_the_interpolant_matches_finite_differences(oracle):
    """On the config-0 tables: central differences of orc_tricubic (inside one cell) against orc_tricubic_grad."""
    O = oracle
    cfg = W.config(0, n=1, T=1e-6)
    fd = dict(cfg["field"], nquant=1, nodes=cfg["field"]["nodes"][:1])
    f = O.Field(fd)
    rng = np.random.default_rng(6)
    for _ in range(20):
        x = np.array([0.05 + 0.9 * rng.random(), 2 * math.pi * rng.random(), 2 * math.pi / 4 * rng.random()])
        v, g = O.tricubic_grad(f, x)
        assert v == O.tricubic(f, x)[0]
        for d in range(3):
            e = np.zeros(3)
            e[d] = 1e-6
            fdiff = (O.tricubic(f, x + e)[0] - O.tricubic(f, x - e)[0]) / 2e-6
            assert abs(fdiff - g[d]) <= 1e-6 * max(1.0, abs(g[d])), (d, fdiff, g[d])
