"""CPU ORACLE for the Chebyshev-filter hot path of DFT-FE (arxiv 2203.07820).  TEST INFRASTRUCTURE ONLY.

This file is a plain, slow, obviously-correct float64 NumPy statement of what the path computes, written
from the paper (citations are `PAPER.md:<line>` = /root/reference/PAPER.md plus the section / equation).
It shares NO code with the CUDA path (`paper_2203_07820_b200/`): its own GLL / Gauss tables, its own shape
functions, its own cell matrices, its own loops.  Only `tests/`, `__graft_entry__.smoke()` and `bench.py`'s
`cpu_baseline` / `--impl reference` leg may import it; the product never does.

What the path computes:

    H~ = M^-1/2 ( 1/2 K + V + sum_a C_a D_a C_a^T ) M^-1/2          Eq. 30 (terms 1-2), 33, 34
    Y  = T_m((H~ - c)/e) X / T_m((a0 - c)/e),  e=(b-a)/2, c=(b+a)/2   Eq. 37 + scaled form of ref. [86]

The cell-level batched form (Eq. 47) and Algorithm 4 are exact
re-bracketings of that global product, so the oracle follows them literally:  extraction -> per-cell dense
product -> assembly, and  C^T X -> assemble P -> scale by D -> C P -> assemble.

Parity pins (tests/test_oracle_*.py, all `-m "not gpu"`): every function below is pinned to a closed form,
an invariant, a textbook/library special case or brute force -- see DESIGN.md Sec. 6.  Parity unpinned: none.

Readings of the paper taken here: U1 scaled recurrence, U2 (p+2)^3 Gauss points for K
and V, U3 P_Ip = N_j N_k, U4 M^-1/2 applied at the vector level, U5 h_lp = D, U6 x-fastest orderings and
trilinear cells.
"""
from __future__ import annotations

from dataclasses import dataclass
from typing import Optional

import numpy as np

# ---------------------------------------------------------------------------------------------------------
# 1-D tables
# ---------------------------------------------------------------------------------------------------------


def legendre(n: int, x):
    """(P_n(x), P_n'(x)) by the three-term recurrence (k+1)P_{k+1} = (2k+1) x P_k - k P_{k-1}."""
    x = np.asarray(x, dtype=np.float64)
    p0, p1 = np.ones_like(x), x.copy()
    if n == 0:
        return p0, np.zeros_like(x)
    for k in range(1, n):
        p0, p1 = p1, ((2 * k + 1) * x * p1 - k * p0) / (k + 1)
    # (1 - x^2) P_n' = n (P_{n-1} - x P_n)
    with np.errstate(divide="ignore", invalid="ignore"):
        dp = n * (p0 - x * p1) / (1 - x * x)
    return p1, dp


def gauss_legendre(nq: int):
    """Gauss-Legendre nodes (ascending) and weights on [-1,1]: roots of P_nq, w = 2/((1-x^2) P_nq'(x)^2)."""
    k = np.arange(1, nq + 1)
    x = -np.cos(np.pi * (k - 0.25) / (nq + 0.5))           # Chebyshev-like initial guess, ascending
    for _ in range(100):
        pn, dpn = legendre(nq, x)
        dx = pn / dpn
        x = x - dx
        if np.max(np.abs(dx)) < 1e-16:
            break
    _, dpn = legendre(nq, x)
    w = 2.0 / ((1 - x * x) * dpn * dpn)
    return x, w


def gauss_lobatto_legendre(p: int):
    """GLL nodes (ascending, p+1 of them) and weights: end points +-1 and the roots of P_p'(x);
    w_i = 2 / (p (p+1) P_p(x_i)^2).  Spectral FE nodes, PAPER.md:301 (Sec. 2.3)."""
    if p < 1:
        raise ValueError("p >= 1")
    x = -np.cos(np.pi * np.arange(p + 1) / p)               # Chebyshev-Gauss-Lobatto initial guess
    xi = x[1:-1].copy()
    for _ in range(100):
        # Newton on q(x) = P_p'(x); q'(x) from Legendre's ODE: (1-x^2) P'' = 2x P' - p(p+1) P
        pn, dpn = legendre(p, xi)
        d2 = (2 * xi * dpn - p * (p + 1) * pn) / (1 - xi * xi)
        dx = dpn / d2
        xi = xi - dx
        if xi.size == 0 or np.max(np.abs(dx)) < 1e-16:
            break
    x[1:-1] = xi
    x[0], x[-1] = -1.0, 1.0
    pn, _ = legendre(p, x)
    w = 2.0 / (p * (p + 1) * pn * pn)
    return x, w


def lagrange_basis(nodes, x):
    """Values and first derivatives of the Lagrange polynomials l_i through `nodes`, at points `x`.
    Returns (L, dL), both [len(x), len(nodes)].  Direct product formula, O(p^3) per point."""
    nodes = np.asarray(nodes, dtype=np.float64)
    x = np.asarray(x, dtype=np.float64)
    n = nodes.size
    L = np.ones((x.size, n))
    dL = np.zeros((x.size, n))
    for i in range(n):
        for j in range(n):
            if j != i:
                L[:, i] *= (x - nodes[j]) / (nodes[i] - nodes[j])
        for k in range(n):
            if k == i:
                continue
            term = np.full(x.size, 1.0 / (nodes[i] - nodes[k]))
            for j in range(n):
                if j != i and j != k:
                    term *= (x - nodes[j]) / (nodes[i] - nodes[j])
            dL[:, i] += term
    return L, dL


# ---------------------------------------------------------------------------------------------------------
# reference-cell tables in 3-D (x fastest: l = a + (p+1)(b + (p+1)c), q = qa + nq1 (qb + nq1 qc))
# ---------------------------------------------------------------------------------------------------------


@dataclass
class RefCell:
    p: int
    gll_x: np.ndarray      # [p+1]
    gll_w: np.ndarray
    gq_x: np.ndarray       # [p+2]
    gq_w: np.ndarray
    N: np.ndarray          # [nq, M_cell]      shape-function values at the Gauss points
    dN: np.ndarray         # [nq, 3, M_cell]   reference-coordinate gradients at the Gauss points
    wq: np.ndarray         # [nq]              tensor-product Gauss weights
    ref_q: np.ndarray      # [nq, 3]
    ref_nodes: np.ndarray  # [M_cell, 3]
    w_nodes: np.ndarray    # [M_cell]          tensor-product GLL weights


def reference_cell(p: int) -> RefCell:
    gx, gw = gauss_lobatto_legendre(p)
    qx, qw = gauss_legendre(p + 2)                           # reading U2: (p+2)^3 Gauss points
    l1, d1 = lagrange_basis(gx, qx)                          # [p+2, p+1]
    n1, nq1 = p + 1, p + 2
    M, nq = n1 ** 3, nq1 ** 3
    N = np.zeros((nq, M))
    dN = np.zeros((nq, 3, M))
    wq = np.zeros(nq)
    ref_q = np.zeros((nq, 3))
    for qc in range(nq1):
        for qb in range(nq1):
            for qa in range(nq1):
                q = qa + nq1 * (qb + nq1 * qc)
                wq[q] = qw[qa] * qw[qb] * qw[qc]
                ref_q[q] = (qx[qa], qx[qb], qx[qc])
                for c in range(n1):
                    for b in range(n1):
                        for a in range(n1):
                            l = a + n1 * (b + n1 * c)
                            N[q, l] = l1[qa, a] * l1[qb, b] * l1[qc, c]
                            dN[q, 0, l] = d1[qa, a] * l1[qb, b] * l1[qc, c]
                            dN[q, 1, l] = l1[qa, a] * d1[qb, b] * l1[qc, c]
                            dN[q, 2, l] = l1[qa, a] * l1[qb, b] * d1[qc, c]
    ref_nodes = np.zeros((M, 3))
    w_nodes = np.zeros(M)
    for c in range(n1):
        for b in range(n1):
            for a in range(n1):
                l = a + n1 * (b + n1 * c)
                ref_nodes[l] = (gx[a], gx[b], gx[c])
                w_nodes[l] = gw[a] * gw[b] * gw[c]
    return RefCell(p, gx, gw, qx, qw, N, dN, wq, ref_q, ref_nodes, w_nodes)


def trilinear_jacobian(vertices, ref_pts):
    """Jacobian J[pt, i, d] = d x_i / d xi_d of the trilinear map of one cell (vertices [8,3], vertex
    v = vx + 2 vy + 4 vz) at reference points [npt, 3]."""
    J = np.zeros((ref_pts.shape[0], 3, 3))
    for v in range(8):
        s = [2 * ((v >> d) & 1) - 1 for d in range(3)]
        f = [(1 + s[d] * ref_pts[:, d]) / 2 for d in range(3)]
        df = [s[d] / 2.0 for d in range(3)]
        grads = [df[0] * f[1] * f[2], f[0] * df[1] * f[2], f[0] * f[1] * df[2]]
        for i in range(3):
            for d in range(3):
                J[:, i, d] += vertices[v, i] * grads[d]
    return J


# ---------------------------------------------------------------------------------------------------------
# the operator
# ---------------------------------------------------------------------------------------------------------


@dataclass
class Operator:
    p: int
    n_cells: int
    n_dofs: int
    cell_dofs: np.ndarray              # [n_cells, M_cell]
    M: np.ndarray                      # [n_dofs]     diagonal GLL mass matrix
    He: np.ndarray                     # [n_cells, M_cell, M_cell]   1/2 K^e + V^e   (NOT Loewdin-scaled)
    n_proj: int
    D: np.ndarray                      # [n_proj]
    proj_cell_ptr: np.ndarray          # CSR projector -> cells
    proj_cell_idx: np.ndarray
    Cc: np.ndarray                     # [nnz, M_cell]  C^c_{l,j} for the (j, c) pair k of the CSR


def mass_diagonal(p, cell_dofs, cell_vertices, n_dofs, ref: Optional[RefCell] = None):
    """M_g = sum over cells containing g of  w_a w_b w_c det J(node):  the overlap matrix integrated with
    the GLL rule whose points coincide with the FE nodes, which makes it diagonal.  PAPER.md:336."""
    ref = ref or reference_cell(p)
    M = np.zeros(n_dofs)
    for c in range(cell_dofs.shape[0]):
        J = trilinear_jacobian(cell_vertices[c], ref.ref_nodes)
        detJ = np.linalg.det(J)
        if np.any(detJ <= 0):
            raise ValueError(f"cell {c}: non-positive Jacobian")
        M[cell_dofs[c]] += ref.w_nodes * detJ              # dofs are distinct inside one cell
    return M


def cell_hamiltonian(ref: RefCell, vertices, veff_q):
    """H^e = 1/2 K^e + V^e for one cell (Eq. 30 terms 1-2; quadrature form Eq. 40,
    PAPER.md:462, with P_Ip = N_j(q_p) N_k(q_p), reading U3):
        K^e_jk = sum_q w_q detJ_q (J_q^-T grad N_j)(q) . (J_q^-T grad N_k)(q)
        V^e_jk = sum_q w_q detJ_q V(q) N_j(q) N_k(q)."""
    J = trilinear_jacobian(vertices, ref.ref_q)              # [nq, 3, 3]
    detJ = np.linalg.det(J)
    if np.any(detJ <= 0):
        raise ValueError("non-positive Jacobian")
    Jinv = np.linalg.inv(J)                                  # Jinv[q, d, i] = d xi_d / d x_i
    # physical gradient of N_l: g[q, i, l] = sum_d Jinv[q, d, i] dN[q, d, l]
    g = np.einsum("qdi,qdl->qil", Jinv, ref.dN)
    wj = ref.wq * detJ
    K = np.einsum("q,qij,qik->jk", wj, g, g, optimize=True)
    V = (ref.N * (wj * veff_q)[:, None]).T @ ref.N
    return 0.5 * K + V, K, V


def projector_cell_vector(ref: RefCell, vertices, chi_q):
    """C^c_{l} = sum_q w_q detJ_q chi(q) N_l(q)   (Eq. 33; Gamma point: phase factors 1)."""
    detJ = np.linalg.det(trilinear_jacobian(vertices, ref.ref_q))
    return ref.N.T @ (ref.wq * detJ * chi_q)


def build_operator(p, cell_dofs, cell_vertices, n_dofs, veff_q, n_proj=0, D=None, proj_cell_ptr=None,
                   proj_cell_idx=None, chi_q=None) -> Operator:
    ref = reference_cell(p)
    n_cells, m_cell = cell_dofs.shape
    assert m_cell == (p + 1) ** 3
    for c in range(n_cells):
        if np.unique(cell_dofs[c]).size != m_cell:
            raise ValueError(f"cell {c}: repeated dof inside one cell")
    M = mass_diagonal(p, cell_dofs, cell_vertices, n_dofs, ref)
    He = np.zeros((n_cells, m_cell, m_cell))
    for c in range(n_cells):
        He[c] = cell_hamiltonian(ref, cell_vertices[c], veff_q[c])[0]
    if n_proj:
        nnz = int(proj_cell_ptr[-1])
        Cc = np.zeros((nnz, m_cell))
        for j in range(n_proj):
            for k in range(int(proj_cell_ptr[j]), int(proj_cell_ptr[j + 1])):
                Cc[k] = projector_cell_vector(ref, cell_vertices[proj_cell_idx[k]], chi_q[k])
        return Operator(p, n_cells, n_dofs, cell_dofs, M, He, n_proj, np.asarray(D, dtype=np.float64),
                        np.asarray(proj_cell_ptr), np.asarray(proj_cell_idx), Cc)
    return Operator(p, n_cells, n_dofs, cell_dofs, M, He, 0, np.zeros(0), np.zeros(1, dtype=np.int64),
                    np.zeros(0, dtype=np.int32), np.zeros((0, m_cell)))


def operator_from_workload(wl) -> Operator:
    return build_operator(wl.p, wl.cell_dofs, wl.cell_vertices, wl.n_dofs, wl.veff_q, wl.n_proj, wl.D,
                          wl.proj_cell_ptr, wl.proj_cell_idx, wl.chi_q)


def apply_H(op: Operator, X):
    """Y = H~ X for a block X [n_dofs, B] of Loewdin-space vectors (Eq. 34).

    Local part, Eq. 47: (i) extraction X -> X^c, (ii) H^c X^c, (iii) assembly.
    Non-local part, Algorithm 4: 1 extraction, 2 P^c = C^cT X^c, 3 P = ASEMB_NLP{P^c},
    4 scale by h_lp (= D, reading U5), 5 Y^c = C^c P^c, 6 ASEMB_FEM."""
    X = np.asarray(X, dtype=np.float64)
    if X.ndim == 1:
        return apply_H(op, X[:, None])[:, 0]
    s = 1.0 / np.sqrt(op.M)
    U = s[:, None] * X                                        # M^-1/2 X (reading U4)
    W = np.zeros_like(U)
    for c in range(op.n_cells):
        g = op.cell_dofs[c]
        W[g] += op.He[c] @ U[g]                               # extraction, dense product, assembly
    if op.n_proj:
        P = np.zeros((op.n_proj, X.shape[1]))
        for j in range(op.n_proj):
            for k in range(int(op.proj_cell_ptr[j]), int(op.proj_cell_ptr[j + 1])):
                g = op.cell_dofs[op.proj_cell_idx[k]]
                P[j] += op.Cc[k] @ U[g]                       # Alg. 4 steps 1-3
        P *= op.D[:, None]                                    # step 4
        for j in range(op.n_proj):
            for k in range(int(op.proj_cell_ptr[j]), int(op.proj_cell_ptr[j + 1])):
                g = op.cell_dofs[op.proj_cell_idx[k]]
                W[g] += np.outer(op.Cc[k], P[j])              # steps 5-6
    return s[:, None] * W


# ---------------------------------------------------------------------------------------------------------
# k-point variant (periodic part u_k of a Bloch wavefunction, Eq. 2-3): complex Hermitian operator
# ---------------------------------------------------------------------------------------------------------


@dataclass
class OperatorK:
    """H~^k = M^-1/2 H^k M^-1/2 with (Eq. 30; Eq. 33)
        H^k_jl = 1/2 int grad N_j . grad N_l + int (V_eff + 1/2 |k|^2) N_j N_l - i int k . (N_j grad N_l)
                 + sum_p C^k_pj h_p conj(C^k_pl),     C^k_pj = int sum_r e^{-i k.(x - L_r)} chi_p(x, R_a + L_r) N_j(x) dx.
    Stored per cell: He = 1/2 K^e + V^e + 1/2 |k|^2 M_G^e (real symmetric), Ae_jl = sum_q w detJ N_j(q) (k . grad N_l)(q)
    (real, antisymmetric after assembly), and the complex projector vectors Cc = Cr + i Ci."""
    base: Operator                     # carries p, cell_dofs, M, He (incl. the 1/2 |k|^2 term), D, projector CSR, Cc = Cr
    kvec: np.ndarray                   # [3]
    Ae: np.ndarray                     # [n_cells, M_cell, M_cell]
    Ci: np.ndarray                     # [nnz, M_cell]   imaginary parts of the projector vectors


def cell_k_term(ref: RefCell, vertices, kvec):
    """Ae_jl = sum_q w_q detJ_q N_j(q) (k . grad_x N_l)(q): the last term of Eq. 30 without its factor -i."""
    J = trilinear_jacobian(vertices, ref.ref_q)
    detJ = np.linalg.det(J)
    Jinv = np.linalg.inv(J)
    g = np.einsum("qdi,qdl->qil", Jinv, ref.dN)              # physical gradients [nq, 3, M_cell]
    kg = np.einsum("i,qil->ql", np.asarray(kvec, dtype=np.float64), g)
    return (ref.N * (ref.wq * detJ)[:, None]).T @ kg


def build_operator_k(p, cell_dofs, cell_vertices, n_dofs, veff_q, kvec, n_proj=0, D=None, proj_cell_ptr=None,
                     proj_cell_idx=None, chi_q=None, chi_q_im=None) -> OperatorK:
    """chi_q + i chi_q_im are the samples of sum_r e^{-i k.(x - L_r)} chi(x, R_a + L_r) at the Gauss points."""
    kvec = np.asarray(kvec, dtype=np.float64)
    base = build_operator(p, cell_dofs, cell_vertices, n_dofs, veff_q + 0.5 * float(kvec @ kvec), n_proj, D,
                          proj_cell_ptr, proj_cell_idx, chi_q)
    ref = reference_cell(p)
    Ae = np.zeros_like(base.He)
    for c in range(base.n_cells):
        Ae[c] = cell_k_term(ref, cell_vertices[c], kvec)
    Ci = np.zeros_like(base.Cc)
    if n_proj and chi_q_im is not None:
        for j in range(n_proj):
            for k in range(int(proj_cell_ptr[j]), int(proj_cell_ptr[j + 1])):
                Ci[k] = projector_cell_vector(ref, cell_vertices[proj_cell_idx[k]], chi_q_im[k])
    return OperatorK(base, kvec, Ae, Ci)


def apply_H_k(opk: OperatorK, X):
    """Y = H~^k X for a complex block X [n_dofs, B], cell by cell as apply_H (Eq. 47, Alg. 4), written on the real and
    imaginary parts:  (He - i Ae)(Ur + i Ui) = (He Ur + Ae Ui) + i (He Ui - Ae Ur);  P = conj(C)^T U;  W += C (D P)."""
    op = opk.base
    X = np.asarray(X, dtype=np.complex128)
    if X.ndim == 1:
        return apply_H_k(opk, X[:, None])[:, 0]
    s = 1.0 / np.sqrt(op.M)
    Ur, Ui = s[:, None] * X.real, s[:, None] * X.imag
    Wr, Wi = np.zeros_like(Ur), np.zeros_like(Ui)
    for c in range(op.n_cells):
        g = op.cell_dofs[c]
        Wr[g] += op.He[c] @ Ur[g] + opk.Ae[c] @ Ui[g]
        Wi[g] += op.He[c] @ Ui[g] - opk.Ae[c] @ Ur[g]
    if op.n_proj:
        Pr = np.zeros((op.n_proj, X.shape[1]))
        Pi = np.zeros((op.n_proj, X.shape[1]))
        for j in range(op.n_proj):
            for k in range(int(op.proj_cell_ptr[j]), int(op.proj_cell_ptr[j + 1])):
                g = op.cell_dofs[op.proj_cell_idx[k]]
                Pr[j] += op.Cc[k] @ Ur[g] + opk.Ci[k] @ Ui[g]        # conj(C) . U
                Pi[j] += op.Cc[k] @ Ui[g] - opk.Ci[k] @ Ur[g]
        Pr *= op.D[:, None]
        Pi *= op.D[:, None]
        for j in range(op.n_proj):
            for k in range(int(op.proj_cell_ptr[j]), int(op.proj_cell_ptr[j + 1])):
                g = op.cell_dofs[op.proj_cell_idx[k]]
                Wr[g] += np.outer(op.Cc[k], Pr[j]) - np.outer(opk.Ci[k], Pi[j])
                Wi[g] += np.outer(op.Cc[k], Pi[j]) + np.outer(opk.Ci[k], Pr[j])
    return s[:, None] * (Wr + 1j * Wi)


def chebyshev_filter_k(opk: OperatorK, X, m: int, a: float, b: float, a0: float):
    """chebyshev_filter for the complex Hermitian H~^k (same scaled recurrence, real scalars)."""
    if m < 1 or not (a0 <= a < b):
        raise ValueError("need m >= 1 and a0 <= a < b")
    X = np.asarray(X, dtype=np.complex128)
    e, c = (b - a) / 2, (b + a) / 2
    sigma1 = e / (a0 - c)
    sigma = sigma1
    Ym2 = X
    Ym1 = (sigma1 / e) * (apply_H_k(opk, X) - c * X)
    for _ in range(2, m + 1):
        sigma_new = 1.0 / (2.0 / sigma1 - sigma)
        Y = (2 * sigma_new / e) * (apply_H_k(opk, Ym1) - c * Ym1) - (sigma * sigma_new) * Ym2
        Ym2, Ym1, sigma = Ym1, Y, sigma_new
    return Ym1


def chebyshev_filter(op: Operator, X, m: int, a: float, b: float, a0: float):
    """Degree-m scaled Chebyshev filter (Eq. 37, in the scaled three-term form of ref. [86]
    (Zhou, Saad, Tiago, Chelikowsky); reading U1):

        e = (b-a)/2, c = (b+a)/2, sigma_1 = e/(a0-c)
        Y_1 = (sigma_1/e) (H~ X - c X)
        sigma_k = 1/(2/sigma_1 - sigma_{k-1});  Y_k = (2 sigma_k/e)(H~ Y_{k-1} - c Y_{k-1}) - sigma_{k-1} sigma_k Y_{k-2}

    which equals T_m((H~-c)/e) X / T_m((a0-c)/e)."""
    if m < 1 or not (a0 <= a < b):
        raise ValueError("need m >= 1 and a0 <= a < b")
    X = np.asarray(X, dtype=np.float64)
    e, c = (b - a) / 2, (b + a) / 2
    sigma1 = e / (a0 - c)
    sigma = sigma1
    Ym2 = X
    Ym1 = (sigma1 / e) * (apply_H(op, X) - c * X)
    for _ in range(2, m + 1):
        sigma_new = 1.0 / (2.0 / sigma1 - sigma)
        Y = (2 * sigma_new / e) * (apply_H(op, Ym1) - c * Ym1) - (sigma * sigma_new) * Ym2
        Ym2, Ym1, sigma = Ym1, Y, sigma_new
    return Ym1


# ---------------------------------------------------------------------------------------------------------
# harness-level helpers (bounds a0, a, b and the Rayleigh-Ritz parity measure; reading U7)
# ---------------------------------------------------------------------------------------------------------


def lanczos_upper_bound(op: Operator, v0, k: int = 20):
    """k-step Lanczos on H~ from start vector v0; returns (upper bound lambda_max(T_k) + |f_k|, lambda_min(T_k)).
    The safeguarded estimator used with Chebyshev filtering in ref. [86]."""
    n = op.n_dofs
    v = np.asarray(v0, dtype=np.float64) / np.linalg.norm(v0)
    alpha, beta = [], []
    v_prev = np.zeros(n)
    f = apply_H(op, v)
    a_ = float(f @ v)
    f = f - a_ * v
    alpha.append(a_)
    for _ in range(1, k):
        b_ = float(np.linalg.norm(f))
        if b_ < 1e-14:
            break
        v_prev, v = v, f / b_
        f = apply_H(op, v) - b_ * v_prev
        a_ = float(f @ v)
        f = f - a_ * v
        alpha.append(a_)
        beta.append(b_)
    T = np.diag(alpha) + np.diag(beta, 1) + np.diag(beta, -1)
    ev = np.linalg.eigvalsh(T)
    return float(ev[-1] + np.linalg.norm(f)), float(ev[0])


def rayleigh_ritz(op: Operator, Y, HY=None, rel_cut: float = 1e-12):
    """Ritz values of H~ in span(Y) (Algorithm 2: S = Y^T Y, H^ = Y^T H~ Y, generalised
    eigenproblem), after column normalisation; directions with S-eigenvalue < rel_cut * max are discarded."""
    Y = np.asarray(Y, dtype=np.float64)
    Y = Y / np.linalg.norm(Y, axis=0, keepdims=True)
    HY = apply_H(op, Y) if HY is None else HY
    S = Y.T @ Y
    Hh = Y.T @ HY
    Hh = 0.5 * (Hh + Hh.T)
    w, Q = np.linalg.eigh(S)
    keep = w > rel_cut * w[-1]
    Qk = Q[:, keep] / np.sqrt(w[keep])[None, :]
    return np.linalg.eigvalsh(Qk.T @ Hh @ Qk)


def projection_matrices(op: Operator, Y):
    """Algorithm 2 step 1 (RRGEP-OP) written out: the overlap matrix S = Y^T Y (step 1a) and the
    projected Hamiltonian H^ = Y^T (H~ Y) (step 1b) of a block Y [n_dofs, N]; no normalisation, no symmetrisation."""
    Y = np.asarray(Y, dtype=np.float64)
    return Y.T @ Y, Y.T @ apply_H(op, Y)


def overlap_mixed(Y, block: int):
    """Mixed-precision overlap matrix of Sec. 3.2 / 4.4.1: "the diagonal block entries of
    overlap matrix S in RRGEP-O are evaluated in FP64 arithmetic while the off-diagonal entries are computed in FP32
    arithmetic".  Blocks are the `block`-wide column blocks of the blocked products; an FP32 block is
    the product of the operands rounded to FP32, accumulated in FP32 (numpy float32 matmul), returned in FP64."""
    Y = np.asarray(Y, dtype=np.float64)
    N = Y.shape[1]
    Y32 = Y.astype(np.float32)
    S = (Y32.T @ Y32).astype(np.float64)
    for j0 in range(0, N, block):
        j1 = min(N, j0 + block)
        S[j0:j1, j0:j1] = Y[:, j0:j1].T @ Y[:, j0:j1]
    return S


def projected_hamiltonian_mixed(Y, HY, n_oc: int):
    """Mixed-precision projected Hamiltonian of Eq. 38-39: with the split Psi_f = [Psi^oc Psi^fr]
    (the first n_oc and the remaining columns), the oc-oc, oc-fr and fr-oc blocks of H^ = Psi_f^T (H~ Psi_f) are
    FP32 products, the fr-fr block is an FP64 product.  HY = H~ Y is given (FP64)."""
    Y = np.asarray(Y, dtype=np.float64)
    HY = np.asarray(HY, dtype=np.float64)
    Hh = (Y.astype(np.float32).T @ HY.astype(np.float32)).astype(np.float64)
    Hh[n_oc:, n_oc:] = Y[:, n_oc:].T @ HY[:, n_oc:]
    return Hh


def cholesky_inverse(S):
    """Algorithm 2 step 2a: Cholesky factor S = L L^T (lower) and its inverse L^-1, by the textbook
    column (Cholesky-Banachiewicz) recursion and forward substitution -- plain loops, no LAPACK."""
    S = np.asarray(S, dtype=np.float64)
    N = S.shape[0]
    L = np.zeros((N, N))
    for j in range(N):
        d = S[j, j] - L[j, :j] @ L[j, :j]
        if not d > 0.0:
            raise np.linalg.LinAlgError("matrix is not positive definite")
        L[j, j] = np.sqrt(d)
        L[j + 1:, j] = (S[j + 1:, j] - L[j + 1:, :j] @ L[j, :j]) / L[j, j]
    Linv = np.zeros((N, N))
    for i in range(N):                       # row i of L^-1 from L L^-1 = I
        e = np.zeros(N)
        e[i] = 1.0
        Linv[i] = (e - L[i, :i] @ Linv[:i]) / L[i, i]
    return L, Linv


def orthonormal_basis_mixed(Y, LinvT):
    """Mixed-precision RRGEP-ST-O: Psi^o = SP[Psi_f (L^-T)_od] + DP[Psi_f (L^-T)_d], with (L^-T)_d the
    diagonal and (L^-T)_od the off-diagonal entries of L^-T: the FP32 product plus an FP64 column scaling."""
    Y = np.asarray(Y, dtype=np.float64)
    d = np.diag(LinvT).copy()
    od = LinvT - np.diag(d)
    return (Y.astype(np.float32) @ od.astype(np.float32)).astype(np.float64) + Y * d[None, :]


def rayleigh_ritz_gep(S, Hh, n_fr: int):
    """Algorithm 2 step 2 (RRGEP-D): Cholesky S = L L^T, standard problem (L^-1 H^ L^-T) Q' = Q' D,
    the n_fr HIGHEST eigenpairs, Q_fr = L^-T Q'_fr.  Returns (D_fr ascending, Q_fr, L^-1)."""
    L, Linv = cholesky_inverse(0.5 * (S + S.T))
    A = Linv @ (0.5 * (Hh + Hh.T)) @ Linv.T
    ev, Qp = np.linalg.eigh(0.5 * (A + A.T))
    return ev[-n_fr:], Linv.T @ Qp[:, -n_fr:], Linv


def ritz_values_of_block(Y, HY, rel_cut: float = 1e-12):
    """Same as rayleigh_ritz but for a given pair (Y, H~Y) (used to compare GPU and oracle blocks with the
    SAME H~Y provider).  Columns are normalised with the norms of Y."""
    nrm = np.linalg.norm(Y, axis=0, keepdims=True)
    Y, HY = Y / nrm, HY / nrm
    S = Y.T @ Y
    Hh = Y.T @ HY
    Hh = 0.5 * (Hh + Hh.T)
    w, Q = np.linalg.eigh(S)
    keep = w > rel_cut * w[-1]
    Qk = Q[:, keep] / np.sqrt(w[keep])[None, :]
    return np.linalg.eigvalsh(Qk.T @ Hh @ Qk)


def apply_H_rows(wl, M, X, rows):
    """Rows `rows` of Y = H~ X computed ONE BY ONE from the definition, without building the whole operator
    (for spot checks at sizes where `build_operator` takes minutes).  `wl` carries the raw inputs (p, cell_dofs,
    cell_vertices, veff_q and the projector CSR / chi_q), `M` is `mass_diagonal(...)`.

        Y[g] = M_g^-1/2 ( sum_{(c,l): dof(c,l)=g} ( H^c[l,:] U^c + sum_{j on c} C^c_{l,j} D_j P_j ) ),  U = M^-1/2 X,
        P_j = sum_{c' in supp(j)} C^{c'}_{:,j} . U^{c'}

    i.e. Eq. 47 and Algorithm 4 restricted to the cells that contain g.
    Pinned in tests/test_oracle_filter.py against `apply_H` (itself pinned to the brute-force dense operator)."""
    X = np.asarray(X, dtype=np.float64)
    ref = reference_cell(wl.p)
    s = 1.0 / np.sqrt(M)
    out = np.zeros((len(rows), X.shape[1]))
    # projector -> cells lists, and cell -> (projector, CSR position) lists for the cells we touch
    P_cache = {}

    def P_of(j):
        if j not in P_cache:
            acc = np.zeros(X.shape[1])
            for k in range(int(wl.proj_cell_ptr[j]), int(wl.proj_cell_ptr[j + 1])):
                c2 = int(wl.proj_cell_idx[k])
                g2 = wl.cell_dofs[c2]
                Cv = projector_cell_vector(ref, wl.cell_vertices[c2], wl.chi_q[k])
                acc += Cv @ (s[g2, None] * X[g2])
            P_cache[j] = acc
        return P_cache[j]

    for r, g in enumerate(rows):
        cells, locs = np.nonzero(wl.cell_dofs == g)
        acc = np.zeros(X.shape[1])
        for c, l in zip(cells, locs):
            gd = wl.cell_dofs[c]
            He = cell_hamiltonian(ref, wl.cell_vertices[c], wl.veff_q[c])[0]
            acc += He[l] @ (s[gd, None] * X[gd])
            if wl.n_proj:
                for j in range(wl.n_proj):
                    k0, k1 = int(wl.proj_cell_ptr[j]), int(wl.proj_cell_ptr[j + 1])
                    hit = np.nonzero(wl.proj_cell_idx[k0:k1] == c)[0]
                    if hit.size:
                        Cv = projector_cell_vector(ref, wl.cell_vertices[c], wl.chi_q[k0 + int(hit[0])])
                        acc += Cv[l] * wl.D[j] * P_of(j)
        out[r] = s[g] * acc
    return out
