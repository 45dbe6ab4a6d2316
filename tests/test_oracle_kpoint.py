"""Pins of the oracle's k-point variant (complex Hermitian H~^k; Eq. 30 k-terms PAPER.md:309-311, Eq. 33 PAPER.md:326,
Bloch form Eq. 2-3).  `-m "not gpu"`.

 * brute force: dense H~^k from a GLOBAL double loop over basis-function pairs (tests/_bruteforce.py), periodic and
   not, distorted cells, with complex projectors;
 * Hermitian; k = 0 reproduces the real operator bit for bit (zero imaginary part);
 * V = 0 on the periodic cube: the nodal interpolant of a plane wave e^{iG.x} has Rayleigh quotient 1/2 |k + G|^2 to
   spectral accuracy, and is an approximate eigenvector;
 * filter: every eigenpair of the dense Hermitian H~^k is mapped to T_m((lambda - c)/e) / T_m((a0 - c)/e) v.
"""
import numpy as np
import pytest

from oracle import chfsi_oracle as orc
from _bruteforce import cheb_T, dense_operator
from workloads.generate import make_workload

KV = np.array([0.21, -0.13, 0.34])


def dense_from_apply(opk, n):
    E = np.eye(n, dtype=np.complex128)
    return orc.apply_H_k(opk, E)


def opk_from_workload(wl):
    return orc.build_operator_k(wl.p, wl.cell_dofs, wl.cell_vertices, wl.n_dofs, wl.veff_q, wl.kvec, wl.n_proj, wl.D,
                                wl.proj_cell_ptr, wl.proj_cell_idx, wl.chi_q, wl.chi_q_im)


@pytest.mark.parametrize("kw", [
    dict(n=2, p=2, L=4.0, periodic=True, mesh_jitter=0.0, r_cut=1.9),
    dict(n=2, p=3, L=4.0, periodic=True, mesh_jitter=0.12, r_cut=1.9),
    dict(n=3, p=2, L=6.0, periodic=False, mesh_jitter=0.1, r_cut=2.5),
])
def test_k_operator_equals_the_brute_force_dense_operator_and_is_hermitian(kw):
    wl = make_workload(None, atoms_per_side=1, n_gaussians=0, nonlocal_=True, smooth_field=0.05, seed_base=31, kvec=KV, **kw)
    opk = opk_from_workload(wl)
    H = dense_from_apply(opk, wl.n_dofs)
    ref = dense_operator(wl.p, wl.cell_dofs, wl.cell_vertices, wl.n_dofs, wl.veff_q, wl.n_proj, wl.D, wl.proj_cell_ptr,
                         wl.proj_cell_idx, wl.chi_q, kvec=KV, chi_q_im=wl.chi_q_im)["Ht"]
    scale = np.max(np.abs(ref))
    assert np.max(np.abs(H - ref)) <= 1e-12 * scale
    if kw["periodic"]:
        assert np.max(np.abs(H - H.conj().T)) <= 1e-12 * scale          # Hermitian on the periodic cell
    assert np.max(np.abs(H.imag)) > 1e-3 * scale                         # the k-terms are really there
    # the sign of the -i k.grad term matters: the conjugate operator is a different one
    assert np.max(np.abs(H.conj() - ref)) > 1e-3 * scale


def test_k_zero_reproduces_the_real_operator_bit_for_bit():
    wl = make_workload(None, n=3, p=3, L=6.0, atoms_per_side=1, n_gaussians=0, nonlocal_=True, smooth_field=0.05,
                       seed_base=32, kvec=[0.0, 0.0, 0.0])
    opk = opk_from_workload(wl)
    op = orc.operator_from_workload(wl)
    rng = np.random.default_rng(1)
    X = rng.standard_normal((wl.n_dofs, 5))
    Yk = orc.apply_H_k(opk, X + 0j)
    assert np.array_equal(Yk.real, orc.apply_H(op, X)) and np.all(Yk.imag == 0.0)
    Z = X + 1j * rng.standard_normal(X.shape)
    Yz = orc.apply_H_k(opk, Z)
    assert np.array_equal(Yz.real, orc.apply_H(op, Z.real)) and np.array_equal(Yz.imag, orc.apply_H(op, Z.imag))
    Fk = orc.chebyshev_filter_k(opk, X + 0j, 6, 1.0, 60.0, 0.2)
    assert np.array_equal(Fk.real, orc.chebyshev_filter(op, X, 6, 1.0, 60.0, 0.2))


@pytest.mark.parametrize("p,tol", [(4, 1e-5), (6, 1e-9)])
def test_plane_waves_on_the_empty_periodic_cube(p, tol):
    """V = 0: u = e^{iG.x} is an eigenfunction of H^k with eigenvalue 1/2 |k + G|^2 (Eq. 2-3: the periodic part of a free
    electron).  Its nodal interpolant v = M^{1/2} u has that Rayleigh quotient with spectral accuracy."""
    n, L = 4, 8.0
    wl = make_workload(None, n=n, p=p, L=L, atoms_per_side=0, n_gaussians=0, nonlocal_=False, smooth_field=0.0,
                       seed_base=33, kvec=KV)
    opk = opk_from_workload(wl)
    nd = n * p
    # physical coordinates of the dofs from the cells
    xyz = np.zeros((wl.n_dofs, 3))
    ref = orc.reference_cell(p)
    for c in range(wl.n_cells):
        v0, v7 = wl.cell_vertices[c, 0], wl.cell_vertices[c, 7]
        xyz[wl.cell_dofs[c]] = v0[None, :] + 0.5 * (ref.ref_nodes + 1.0) * (v7 - v0)[None, :]
    xyz = xyz % L
    for G in ([0, 0, 0], [1, 0, 0], [0, -1, 1], [1, 1, -1]):
        Gv = 2 * np.pi / L * np.array(G, dtype=np.float64)
        u = np.exp(1j * (xyz @ Gv))
        v = np.sqrt(opk.base.M) * u
        Hv = orc.apply_H_k(opk, v)
        lam = 0.5 * float((KV + Gv) @ (KV + Gv))
        rq = (np.vdot(v, Hv) / np.vdot(v, v))
        assert abs(rq.imag) <= 1e-12 and abs(rq.real - lam) <= tol * max(1.0, lam), (G, rq, lam)
        assert np.linalg.norm(Hv - lam * v) <= 50 * np.sqrt(tol) * np.linalg.norm(v) * max(1.0, lam)
    # the k-dependence is the physical one: flipping the sign of k changes the G = (1,0,0) eigenvalue
    assert abs(0.5 * np.sum((KV + 2 * np.pi / L * np.array([1, 0, 0])) ** 2) -
               0.5 * np.sum((-KV + 2 * np.pi / L * np.array([1, 0, 0])) ** 2)) > 1e-2


def test_filter_maps_every_eigenpair_of_the_hermitian_operator_to_the_chebyshev_value():
    wl = make_workload(None, n=2, p=3, L=4.0, atoms_per_side=1, n_gaussians=0, nonlocal_=True, smooth_field=0.05,
                       seed_base=34, kvec=KV, r_cut=1.9)
    opk = opk_from_workload(wl)
    H = dense_from_apply(opk, wl.n_dofs)
    H = 0.5 * (H + H.conj().T)
    ev, V = np.linalg.eigh(H)
    b, a, a0 = ev[-1] + 0.5, ev[len(ev) // 4], ev[0] - 0.1
    e, c = (b - a) / 2, (b + a) / 2
    for m in (1, 2, 7):
        F = orc.chebyshev_filter_k(opk, V, m, a, b, a0)
        gain = cheb_T(m, (ev - c) / e) / cheb_T(m, np.array([(a0 - c) / e]))[0]
        assert np.max(np.abs(F - V * gain[None, :])) <= 1e-9 * np.max(np.abs(gain))
