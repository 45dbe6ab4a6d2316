"""Independent brute-force statements of the operator, used ONLY to pin the oracle (tests, CPU).

Nothing here is shared with `oracle/` or with the CUDA library.  Everything is built from
`numpy.polynomial` objects (Legendre series, polynomial roots / derivatives / integrals) and from a *global*
formulation: every global basis function is tabulated at every quadrature point of every cell and the
dense matrix is one big product  H = sum_d (d_d Phi)^T W (d_d Phi)/2 + Phi^T (W V) Phi  (Eq. 30 terms 1-2,
PAPER.md:309), i.e. a double loop over global basis-function pairs, not a cell-by-cell assembly.
"""
from __future__ import annotations

import numpy as np
from numpy.polynomial import legendre as npleg
from numpy.polynomial import polynomial as nppoly


def gll_nodes_weights(p: int):
    """GLL nodes as the roots of (1-x^2) P_p'(x) found by numpy's companion-matrix root finder, weights by
    integrating the Lagrange polynomials exactly (interpolatory quadrature), not by the closed formula."""
    Pp = npleg.Legendre.basis(p)
    inner = np.sort(np.real(Pp.deriv().roots())) if p > 1 else np.zeros(0)
    x = np.concatenate([[-1.0], inner, [1.0]])
    w = np.zeros(p + 1)
    for i in range(p + 1):
        c = lagrange_coeffs(x, i)
        ci = nppoly.polyint(c)
        w[i] = nppoly.polyval(1.0, ci) - nppoly.polyval(-1.0, ci)
    return x, w


def lagrange_coeffs(nodes, i):
    """Monomial coefficients of the i-th Lagrange polynomial through `nodes`."""
    others = np.delete(nodes, i)
    c = nppoly.polyfromroots(others)
    return c / nppoly.polyval(nodes[i], c)


def lagrange_tables(nodes, x):
    """L[k, i] = l_i(x_k), dL[k, i] = l_i'(x_k) from monomial coefficients."""
    n = len(nodes)
    L = np.zeros((len(x), n))
    dL = np.zeros((len(x), n))
    for i in range(n):
        c = lagrange_coeffs(np.asarray(nodes), i)
        L[:, i] = nppoly.polyval(x, c)
        dL[:, i] = nppoly.polyval(x, nppoly.polyder(c))
    return L, dL


def trilinear_map(verts, ref):
    """x(xi) for one cell: verts [8,3] (v = vx + 2vy + 4vz), ref [n,3] in [-1,1]^3."""
    out = np.zeros((ref.shape[0], 3))
    for v in range(8):
        w = np.ones(ref.shape[0])
        for d in range(3):
            bit = (v >> d) & 1
            w = w * ((1 + ref[:, d]) / 2 if bit else (1 - ref[:, d]) / 2)
        out += w[:, None] * verts[v][None, :]
    return out


def jacobian_fd(verts, ref, h=0.25):
    """J[k, i, d] = dx_i/dxi_d by central differences -- exact (up to rounding) for a trilinear map because
    the map is affine in each xi_d separately."""
    J = np.zeros((ref.shape[0], 3, 3))
    for d in range(3):
        e = np.zeros(3)
        e[d] = h
        J[:, :, d] = (trilinear_map(verts, ref + e) - trilinear_map(verts, ref - e)) / (2 * h)
    return J


def dense_operator(p, cell_dofs, cell_vertices, n_dofs, veff_q, n_proj=0, D=None, proj_cell_ptr=None,
                   proj_cell_idx=None, chi_q=None, nq1=None, kvec=None, chi_q_im=None):
    """Dense (M_diag, Hloc, C, H~) for a tiny mesh by the global formulation described in the module
    docstring.  Returns dict with 'M' [n], 'K' [n,n], 'V' [n,n], 'C' [n,n_proj], 'Ht' [n,n].
    With `kvec` the k-point operator of Eq. 30 / 33 is returned as a complex 'Ht':
    H^k = 1/2 K + V + 1/2 |k|^2 M_G - i A_k + C h C^dagger, (A_k)_jl = int N_j k.grad N_l, C complex."""
    nq1 = nq1 or p + 2
    gx, gw = gll_nodes_weights(p)
    qx, qw = npleg.leggauss(nq1)
    L1, d1 = lagrange_tables(gx, qx)
    n1 = p + 1
    n_cells = cell_dofs.shape[0]
    nq = nq1 ** 3
    Phi = np.zeros((n_cells, nq, n_dofs))
    dPhi = np.zeros((n_cells, nq, 3, n_dofs))
    W = np.zeros((n_cells, nq))
    q = np.arange(nq)
    qa, qb, qc = q % nq1, (q // nq1) % nq1, q // (nq1 * nq1)
    ref_q = np.stack([qx[qa], qx[qb], qx[qc]], axis=1)
    wq = qw[qa] * qw[qb] * qw[qc]
    for c in range(n_cells):
        J = jacobian_fd(cell_vertices[c], ref_q)
        detJ = np.linalg.det(J)
        W[c] = wq * detJ
        Jinv = np.linalg.inv(J)
        for l in range(n1 ** 3):
            a, b, cc = l % n1, (l // n1) % n1, l // (n1 * n1)
            g = cell_dofs[c, l]
            val = L1[qa, a] * L1[qb, b] * L1[qc, cc]
            gref = np.stack([d1[qa, a] * L1[qb, b] * L1[qc, cc],
                             L1[qa, a] * d1[qb, b] * L1[qc, cc],
                             L1[qa, a] * L1[qb, b] * d1[qc, cc]], axis=1)          # [nq, 3] d/dxi
            # physical gradient: dN/dx_i = sum_d dN/dxi_d * dxi_d/dx_i
            gphys = np.einsum("qd,qdi->qi", gref, Jinv)
            Phi[c, :, g] += val
            dPhi[c, :, :, g] += gphys
    Phi2 = Phi.reshape(n_cells * nq, n_dofs)
    Wf = W.reshape(-1)
    K = np.zeros((n_dofs, n_dofs))
    for d in range(3):
        G = dPhi[:, :, d, :].reshape(n_cells * nq, n_dofs)
        K += G.T @ (Wf[:, None] * G)
    V = Phi2.T @ ((Wf * veff_q.reshape(-1))[:, None] * Phi2)
    # diagonal mass: GLL quadrature at the nodes
    M = np.zeros(n_dofs)
    l = np.arange(n1 ** 3)
    ref_n = np.stack([gx[l % n1], gx[(l // n1) % n1], gx[l // (n1 * n1)]], axis=1)
    wn = gw[l % n1] * gw[(l // n1) % n1] * gw[l // (n1 * n1)]
    for c in range(n_cells):
        detJ = np.linalg.det(jacobian_fd(cell_vertices[c], ref_n))
        np.add.at(M, cell_dofs[c], wn * detJ)
    C = np.zeros((n_dofs, max(n_proj, 0)))
    for j in range(n_proj):
        for k in range(int(proj_cell_ptr[j]), int(proj_cell_ptr[j + 1])):
            c = int(proj_cell_idx[k])
            C[:, j] += Phi[c].T @ (W[c] * chi_q[k])
    Hloc = 0.5 * K + V
    s = 1 / np.sqrt(M)
    if kvec is not None:
        kvec = np.asarray(kvec, dtype=np.float64)
        MG = Phi2.T @ (Wf[:, None] * Phi2)
        A = np.zeros((n_dofs, n_dofs))
        for d in range(3):
            G = dPhi[:, :, d, :].reshape(n_cells * nq, n_dofs)
            A += kvec[d] * (Phi2.T @ (Wf[:, None] * G))
        Ck = C.astype(np.complex128)
        if n_proj and chi_q_im is not None:
            for j in range(n_proj):
                for k in range(int(proj_cell_ptr[j]), int(proj_cell_ptr[j + 1])):
                    c = int(proj_cell_idx[k])
                    Ck[:, j] += 1j * (Phi[c].T @ (W[c] * chi_q_im[k]))
        Hk = Hloc + 0.5 * float(kvec @ kvec) * MG - 1j * A
        if n_proj:
            Hk = Hk + Ck @ np.diag(np.asarray(D, dtype=np.float64)) @ Ck.conj().T
        return dict(M=M, K=K, V=V, C=Ck, A=A, Ht=s[:, None] * Hk * s[None, :])
    H = Hloc + (C @ np.diag(np.asarray(D, dtype=np.float64)) @ C.T if n_proj else 0.0)
    return dict(M=M, K=K, V=V, C=C, Hloc=Hloc, Ht=s[:, None] * H * s[None, :])


def cheb_T(m: int, t):
    """T_m(t) for real t by the hyperbolic / trigonometric closed forms (not by the recurrence)."""
    t = np.asarray(t, dtype=np.float64)
    out = np.empty_like(t)
    inside = np.abs(t) <= 1
    out[inside] = np.cos(m * np.arccos(t[inside]))
    big = ~inside
    sgn = np.where(t[big] < 0, (-1.0) ** m, 1.0)
    out[big] = sgn * np.cosh(m * np.arccosh(np.abs(t[big])))
    return out
