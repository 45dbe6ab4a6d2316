"""GPU parity of the k-point variant (chfsi_create_k: complex Hermitian H~^k, Eq. 30 k-terms PAPER.md:309-311, Eq. 33
phases PAPER.md:326) against the oracle's apply_H_k / chebyshev_filter_k, through the C ABI.  `-m gpu`.

Tolerances as for the real FP64 path (north_star): relative Frobenius and max-norm error <= 1e-10, Rayleigh-Ritz values of
the filtered subspace within 1e-8 Ha (generalised Hermitian problem, the ORACLE's H~^k on both blocks)."""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu

KV = np.array([0.21, -0.13, 0.34])


def _imports():
    import torch
    from oracle import chfsi_oracle as orc
    from paper_2203_07820_b200 import ChfsiError, Operator
    from workloads.generate import make_workload, random_block
    return torch, orc, Operator, ChfsiError, make_workload, random_block


def opk_from_workload(orc, wl):
    return orc.build_operator_k(wl.p, wl.cell_dofs, wl.cell_vertices, wl.n_dofs, wl.veff_q, wl.kvec, wl.n_proj, wl.D,
                                wl.proj_cell_ptr, wl.proj_cell_idx, wl.chi_q, wl.chi_q_im)


def complex_block(random_block, n_dofs, B, seed):
    return random_block(n_dofs, range(B), seed) + 1j * random_block(n_dofs, range(B), seed + 1)


def assert_close(Y, Yo, tol, what):
    assert Y.shape == Yo.shape and np.all(np.isfinite(Y)), what
    err = float(np.linalg.norm(Y - Yo) / np.linalg.norm(Yo))
    emax = float(np.max(np.abs(Y - Yo)) / np.max(np.abs(Yo)))
    assert err <= tol and emax <= tol, f"{what}: rel Frobenius {err:.3e}, max-norm {emax:.3e} > {tol:g}"


def hermitian_ritz_values(orc, opk, F, rel_cut=1e-12):
    """Algorithm 2 for a complex block: column-normalise, S = F^H F, H^ = F^H H~^k F with the oracle's
    operator, drop S-directions below rel_cut, eigenvalues of the reduced Hermitian problem."""
    F = F / np.linalg.norm(F, axis=0)
    S = F.conj().T @ F
    Hh = F.conj().T @ orc.apply_H_k(opk, F)
    s, U = np.linalg.eigh(S)
    keep = s > rel_cut * s.max()
    T = U[:, keep] / np.sqrt(s[keep])
    return np.linalg.eigvalsh(T.conj().T @ (0.5 * (Hh + Hh.conj().T)) @ T)


CASES = {
    # name: (workload kwargs, complex columns B, degree m)
    "p6_nonlocal_ragged": (dict(n=3, p=6, L=6.0, atoms_per_side=1, n_gaussians=0, nonlocal_=True, smooth_field=0.05,
                                seed_base=77), 20, 6),             # 40 real columns: two 16-column tiles + a ragged one
    "p6_distorted_cells": (dict(n=2, p=6, L=4.0, mesh_jitter=0.15, atoms_per_side=1, n_gaussians=0, nonlocal_=True,
                                smooth_field=0.05, seed_base=78, r_cut=1.9), 12, 5),
    "p3_distorted": (dict(n=3, p=3, L=6.0, mesh_jitter=0.1, atoms_per_side=1, n_gaussians=0, nonlocal_=True,
                          smooth_field=0.05, seed_base=79), 7, 5),
    "p2_nonperiodic": (dict(n=3, p=2, L=6.0, periodic=False, atoms_per_side=1, n_gaussians=0, nonlocal_=True,
                            smooth_field=0.05, seed_base=80, r_cut=2.5), 4, 4),
    "p4_no_projectors": (dict(n=3, p=4, L=6.0, atoms_per_side=1, n_gaussians=3, nonlocal_=False, smooth_field=0.05,
                              seed_base=81), 9, 7),
    # two atoms per side: cells in the overlap of two supports, dofs that two projector groups add to
    "p5_overlapping_supports": (dict(n=4, p=5, L=8.0, atoms_per_side=2, n_gaussians=0, nonlocal_=True, smooth_field=0.05,
                                     seed_base=82, r_cut=2.0), 8, 4),
}

_cache = {}


def oracle_case(name):
    if name in _cache:
        return _cache[name]
    torch, orc, Operator, _, make_workload, random_block = _imports()
    kw, B, m = CASES[name]
    wl = make_workload(None, kvec=KV, **kw)
    opk = opk_from_workload(orc, wl)
    X = complex_block(random_block, wl.n_dofs, B, 11)
    # bounds from the real operator (the k-terms move the spectrum by O(|k| sqrt(lambda_max)) at most): any a0 <= a < b is a
    # valid filter, the comparison is of the polynomial
    oop = orc.operator_from_workload(wl)
    b0, lmin = orc.lanczos_upper_bound(oop, np.random.default_rng(5).standard_normal(wl.n_dofs), 20)
    b = 1.2 * b0 + 1.0
    a0, a = lmin, lmin + 0.1 * (b - lmin)
    Yo = orc.apply_H_k(opk, X)
    Fo = orc.chebyshev_filter_k(opk, X, m, a, b, a0)
    _cache[name] = (wl, opk, X, (a0, a, b), Yo, Fo)
    return _cache[name]


@pytest.mark.parametrize("assembly", [0, 1])
@pytest.mark.parametrize("name", list(CASES))
def test_k_apply_and_filter_match_the_oracle(name, assembly):
    torch, orc, Operator, *_ = _imports()
    _, B, m = CASES[name]
    wl, opk, X, (a0, a, b), Yo, Fo = oracle_case(name)
    op = Operator.from_workload(wl, assembly=assembly)
    assert op.kpoint and op.dtype == torch.complex128
    Xd = torch.tensor(X, dtype=torch.complex128, device="cuda")
    n0 = op.launch_count()
    Y = op.apply_H(Xd).cpu().numpy()
    assert op.launch_count() > n0, "no kernel was launched"
    assert_close(Y, Yo, 1e-10, f"{name} apply_H_k")
    assert np.max(np.abs(Yo.imag)) > 1e-3 * np.max(np.abs(Yo))           # a genuinely complex result
    F = Xd.clone()
    op.chebyshev_filter(F, m, a, b, a0)
    F = F.cpu().numpy()
    assert_close(F, Fo, 1e-10, f"{name} filter m={m}")
    th_g = hermitian_ritz_values(orc, opk, F)
    th_o = hermitian_ritz_values(orc, opk, Fo)
    assert th_g.shape == th_o.shape
    assert np.max(np.abs(th_g - th_o)) <= 1e-8, f"{name}: Ritz values differ by {np.max(np.abs(th_g - th_o)):.3e} Ha"
    op.close()


def test_sign_of_the_k_term_and_of_the_phases_matters():
    """The conjugate operator (k -> -k, phases conjugated) is a different one: the comparison above would not pass with
    a flipped sign anywhere."""
    torch, orc, Operator, *_ = _imports()
    wl, opk, X, _, Yo, _ = oracle_case("p3_distorted")
    Yc = orc.apply_H_k(opk, X.conj()).conj()                              # conj(H) X
    assert np.linalg.norm(Yc - Yo) > 1e-3 * np.linalg.norm(Yo)


def test_k_zero_equals_the_real_operator_on_both_parts():
    torch, orc, Operator, _, make_workload, random_block = _imports()
    kw = dict(n=3, p=6, L=6.0, atoms_per_side=1, n_gaussians=0, nonlocal_=True, smooth_field=0.05, seed_base=77)
    wl0 = make_workload(None, kvec=[0.0, 0.0, 0.0], **kw)
    wlr = make_workload(None, **kw)
    opk, opr = Operator.from_workload(wl0), Operator.from_workload(wlr)
    X = complex_block(random_block, wl0.n_dofs, 16, 3)
    Xd = torch.tensor(X, dtype=torch.complex128, device="cuda")
    Y = opk.apply_H(Xd)
    Yr = opr.apply_H(Xd.real.contiguous())
    Yi = opr.apply_H(Xd.imag.contiguous())
    # (same fields and column arithmetic; the projector term is added by a different kernel: equal to rounding)
    assert float((Y.real - Yr).norm() / Yr.norm()) <= 1e-14 and float((Y.imag - Yi).norm() / Yi.norm()) <= 1e-14
    F = Xd.clone()
    opk.chebyshev_filter(F, 5, 0.4, 300.0, 0.1)
    Fr = Xd.real.contiguous()
    opr.chebyshev_filter(Fr, 5, 0.4, 300.0, 0.1)
    assert float((F.real - Fr).norm() / Fr.norm()) <= 1e-13
    opk.close(); opr.close()


def test_k_filter_is_bit_reproducible_chunked_and_from_the_host():
    torch, orc, Operator, *_ = _imports()
    wl, opk, X, (a0, a, b), _, Fo = oracle_case("p5_overlapping_supports")
    m = CASES["p5_overlapping_supports"][2]
    op = Operator.from_workload(wl)
    Xd = torch.tensor(X, dtype=torch.complex128, device="cuda")
    runs = []
    for _ in range(3):
        F = Xd.clone()
        op.chebyshev_filter(F, m, a, b, a0)
        runs.append(F)
    assert torch.equal(torch.view_as_real(runs[0]), torch.view_as_real(runs[1]))
    assert torch.equal(torch.view_as_real(runs[0]), torch.view_as_real(runs[2]))
    # a chunk of a wider array (ld > B), chunks of 4 complex columns; columns are independent
    wide = torch.full((wl.n_dofs, X.shape[1] + 6), 7.0 + 1.0j, dtype=torch.complex128, device="cuda")
    wide[:, :X.shape[1]] = Xd
    op.chebyshev_filter_chunked(wide[:, :X.shape[1]], 4, m, a, b, a0)
    assert_close(wide[:, :X.shape[1]].cpu().numpy(), Fo, 1e-10, "chunked, ld > B")
    assert bool((wide[:, X.shape[1]:] == 7.0 + 1.0j).all())
    # host entry point
    Xh = np.ascontiguousarray(X)
    op.chebyshev_filter_host(Xh, 8, m, a, b, a0)
    assert_close(Xh, Fo, 1e-10, "host entry point")
    op.close()


def test_k_handle_argument_errors():
    torch, orc, Operator, ChfsiError, make_workload, _ = _imports()
    wl7 = make_workload(None, n=2, p=7, L=4.0, atoms_per_side=1, n_gaussians=2, nonlocal_=False, smooth_field=0.0, seed_base=83,
                        kvec=KV)
    with pytest.raises(ChfsiError) as e:
        Operator.from_workload(wl7)
    assert e.value.code == -5                                             # p = 7: no sum-factorised kernel
    wl = oracle_case("p2_nonperiodic")[0]
    op = Operator.from_workload(wl)
    Y = torch.zeros((wl.n_dofs, 4), dtype=torch.complex128, device="cuda")
    with pytest.raises(ChfsiError) as e:                                  # the Rayleigh-Ritz calls take real blocks only
        import ctypes as C
        from paper_2203_07820_b200 import load_library
        S = torch.zeros((4, 4), dtype=torch.float64, device="cuda")
        rc = load_library().chfsi_overlap_matrix(op._h, C.c_void_p(Y.data_ptr()), 4, 4, C.c_void_p(S.data_ptr()), None)
        op._check(rc)
    assert e.value.code == -5
    with pytest.raises(TypeError):
        op.apply_H(torch.zeros((wl.n_dofs, 4), dtype=torch.float64, device="cuda"))
    op.close()
