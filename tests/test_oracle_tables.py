"""Pins for the oracle's 1-D tables and reference cell (SURVEY.md 8(c) "GLL / Gauss tables").  CPU only."""
import numpy as np
import pytest

from oracle import chfsi_oracle as orc

from _bruteforce import gll_nodes_weights, lagrange_tables


def _read_golden(name):
    import os
    path = os.path.join(os.path.dirname(__file__), "golden", name)
    rows = [l.split("#")[0].split() for l in open(path) if l.split("#")[0].strip()]
    return rows


def test_gll_textbook_values():
    """tests/golden/gll_textbook.txt: closed-form GLL rules for p = 1..4 (Abramowitz & Stegun 25.4.32:
    x = +-1, roots of P_p'; w = 2/(p(p+1)P_p(x)^2)), typed in as exact radicals."""
    for row in _read_golden("gll_textbook.txt"):
        p, i = int(row[0]), int(row[1])
        x_expected, w_expected = eval(row[2]), eval(row[3])          # radicals like sqrt(1/5)
        x, w = orc.gauss_lobatto_legendre(p)
        assert abs(x[i] - x_expected) < 1e-15
        assert abs(w[i] - w_expected) < 1e-15


@pytest.mark.parametrize("p", [1, 2, 3, 4, 5, 6, 7, 8])
def test_gll_exactness_and_independent_construction(p):
    x, w = orc.gauss_lobatto_legendre(p)
    assert x[0] == -1 and x[-1] == 1 and np.all(np.diff(x) > 0)
    assert abs(w.sum() - 2) < 1e-14
    for k in range(0, 2 * p):                                         # exact to degree 2p-1
        exact = 0.0 if k % 2 else 2.0 / (k + 1)
        assert abs(np.sum(w * x ** k) - exact) < 2e-14
    # degree 2p is NOT integrated exactly (otherwise the rule would be Gauss, not Lobatto)
    assert abs(np.sum(w * x ** (2 * p)) - 2.0 / (2 * p + 1)) > 1e-6
    xb, wb = gll_nodes_weights(p)                                     # companion-matrix roots + exact integrals
    assert np.allclose(x, xb, atol=1e-13) and np.allclose(w, wb, atol=1e-13)


@pytest.mark.parametrize("nq", [1, 2, 3, 6, 8, 9, 10])
def test_gauss_legendre_vs_numpy_and_exactness(nq):
    x, w = orc.gauss_legendre(nq)
    xn, wn = np.polynomial.legendre.leggauss(nq)
    assert np.allclose(x, xn, atol=1e-14) and np.allclose(w, wn, atol=1e-14)
    for k in range(0, 2 * nq):                                        # exact to degree 2nq-1 (= 2p+3 for nq=p+2)
        exact = 0.0 if k % 2 else 2.0 / (k + 1)
        assert abs(np.sum(w * x ** k) - exact) < 2e-14


@pytest.mark.parametrize("p", [1, 2, 4, 6])
def test_lagrange_basis(p):
    x, _ = orc.gauss_lobatto_legendre(p)
    L, dL = orc.lagrange_basis(x, x)
    assert np.allclose(L, np.eye(p + 1), atol=1e-13)                   # cardinal property
    pts = np.linspace(-1, 1, 11)
    L, dL = orc.lagrange_basis(x, pts)
    assert np.allclose(L.sum(axis=1), 1, atol=1e-13)                   # partition of unity
    assert np.allclose(dL.sum(axis=1), 0, atol=1e-11)
    for k in range(p + 1):                                             # reproduces monomials and derivatives
        assert np.allclose(L @ x ** k, pts ** k, atol=1e-12)
        assert np.allclose(dL @ x ** k, k * pts ** max(k - 1, 0) if k else 0 * pts, atol=1e-10)
    Lb, dLb = lagrange_tables(x, pts)                                  # monomial-coefficient construction
    assert np.allclose(L, Lb, atol=1e-11) and np.allclose(dL, dLb, atol=1e-9)


def test_reference_cell_orderings():
    """x-fastest orderings (reading U6): l = a + (p+1)(b + (p+1)c), q likewise."""
    p = 2
    ref = orc.reference_cell(p)
    assert ref.N.shape == (64, 27) and ref.dN.shape == (64, 3, 27)
    # node 1 is the second GLL point along x: reference coordinates (0, -1, -1)
    assert np.allclose(ref.ref_nodes[1], [0, -1, -1]) and np.allclose(ref.ref_nodes[3], [-1, 0, -1])
    assert np.allclose(ref.ref_nodes[9], [-1, -1, 0])
    assert ref.ref_q[1][0] > ref.ref_q[0][0] and ref.ref_q[1][1] == ref.ref_q[0][1]
    assert abs(ref.wq.sum() - 8) < 1e-13 and abs(ref.w_nodes.sum() - 8) < 1e-13
    # f(x,y,z) = x + 2y + 3z is in the FE space: interpolation and gradient are exact at the Gauss points
    f = ref.ref_nodes @ np.array([1.0, 2.0, 3.0])
    assert np.allclose(ref.N @ f, ref.ref_q @ np.array([1.0, 2.0, 3.0]), atol=1e-13)
    g = np.einsum("qdl,l->qd", ref.dN, f)
    assert np.allclose(g, np.array([1.0, 2.0, 3.0])[None, :], atol=1e-12)


def test_trilinear_jacobian_affine_and_general():
    rng = np.random.default_rng(0)
    A = np.eye(3) + 0.2 * rng.standard_normal((3, 3))
    corners = np.array([[(v >> d) & 1 for d in range(3)] for v in range(8)], dtype=float) * 2 - 1
    verts = corners @ A.T + 0.3
    pts = rng.uniform(-1, 1, (5, 3))
    J = orc.trilinear_jacobian(verts, pts)
    assert np.allclose(J, A[None], atol=1e-13)                          # affine map: J = A everywhere
    from _bruteforce import jacobian_fd
    verts2 = verts + 0.1 * rng.standard_normal((8, 3))
    assert np.allclose(orc.trilinear_jacobian(verts2, pts), jacobian_fd(verts2, pts), atol=1e-12)
