"""Pins for the oracle's Chebyshev filter, bounds estimators and Rayleigh-Ritz measure: SURVEY.md 8(c).  CPU only.

The filter is a matrix polynomial of H~ (Eq. 37), so on every eigenpair (lambda, v) of the dense
H~ its action is fixed by mathematics alone:  v -> T_m((lambda-c)/e) / T_m((a0-c)/e) v.  The scalar Chebyshev
values are evaluated here by the closed forms cos(m acos t) / cosh(m acosh |t|) -- not by any recurrence -- so a
wrong sign, a dropped term, a swapped sigma index or a wrong normalisation in the oracle's loop fails.
"""
import json
import os

import numpy as np
import pytest

from oracle import chfsi_oracle as orc
from workloads.generate import CONFIGS, SEED_LANCZOS, SEED_RR, load_bounds, make_workload, random_block


def cheb_T(m, t):
    """T_m(t) by the closed forms (no recurrence)."""
    t = np.asarray(t, dtype=np.float64)
    out = np.empty_like(t)
    inside = np.abs(t) <= 1
    out[inside] = np.cos(m * np.arccos(t[inside]))
    big = ~inside
    out[big] = np.cosh(m * np.arccosh(np.abs(t[big]))) * np.where(t[big] < 0, (-1.0) ** m, 1.0)
    return out


def tiny(n=2, p=3, L=4.0, nonlocal_=True, seed=11, smooth=0.05, gauss=True):
    return make_workload(None, n=n, p=p, L=L, atoms_per_side=1 if gauss else 0, n_gaussians=0,
                         nonlocal_=nonlocal_, smooth_field=smooth, seed_base=seed, r_cut=1.5)


@pytest.fixture(scope="module")
def tiny_eig():
    wl = tiny()
    op = orc.operator_from_workload(wl)
    H = orc.apply_H(op, np.eye(op.n_dofs))
    lam, V = np.linalg.eigh(0.5 * (H + H.T))
    return op, lam, V


@pytest.mark.parametrize("m", [1, 2, 3, 8, 15])
def test_filter_acts_on_every_eigenvector_by_the_scalar_chebyshev_value(tiny_eig, m):
    op, lam, V = tiny_eig
    a0 = lam[0] - 0.05
    a = lam[0] + 0.15 * (lam[-1] - lam[0])
    b = lam[-1] + 0.3
    e, c = (b - a) / 2, (b + a) / 2
    gain = cheb_T(m, (lam - c) / e) / cheb_T(m, np.array([(a0 - c) / e]))[0]
    Y = orc.chebyshev_filter(op, V, m, a, b, a0)
    assert np.allclose(Y, V * gain[None, :], rtol=0, atol=1e-11 * np.max(np.abs(gain)))
    # unwanted part of the spectrum (a, b) is damped to |gain| <= 1/T_m(t0), the wanted part is amplified
    assert np.all(np.abs(gain[lam > a]) <= 1.0 / abs(cheb_T(m, np.array([(a0 - c) / e]))[0]) + 1e-15)


def test_component_at_a0_has_gain_one_and_m1_is_the_affine_map(tiny_eig):
    op, lam, V = tiny_eig
    a0, a, b = lam[0], lam[3], lam[-1] + 0.1                    # a0 exactly an eigenvalue
    for m in (1, 4, 9):
        y = orc.chebyshev_filter(op, V[:, :1], m, a, b, a0)
        assert np.allclose(y, V[:, :1], atol=1e-11)
    X = random_block(op.n_dofs, range(3), 5)
    e, c = (b - a) / 2, (b + a) / 2
    Y1 = orc.chebyshev_filter(op, X, 1, a, b, a0)
    assert np.allclose(Y1, (orc.apply_H(op, X) - c * X) / (a0 - c), rtol=1e-13, atol=1e-13)


def test_V0_periodic_cube_constant_mode_closed_form_without_eigh():
    """north_star's check: V_eff = 0 on a periodic cube; v = M^{1/2} 1 is an exact eigenvector with lambda = 0
    (constants are in the null space of K), so the filter returns T_m(-c/e)/T_m((a0-c)/e) v."""
    wl = make_workload(None, n=3, p=3, L=6.0, atoms_per_side=0, n_gaussians=0, nonlocal_=False, smooth_field=0.0,
                       seed_base=3)
    assert np.all(wl.veff_q == 0)
    op = orc.operator_from_workload(wl)
    v = np.sqrt(op.M)[:, None]
    a0, a, b = -0.2, 1.0, 40.0
    e, c = (b - a) / 2, (b + a) / 2
    for m in (1, 6, 13):
        g = cheb_T(m, np.array([(0.0 - c) / e]))[0] / cheb_T(m, np.array([(a0 - c) / e]))[0]
        assert np.allclose(orc.chebyshev_filter(op, v, m, a, b, a0), g * v, rtol=1e-11, atol=1e-12)


def test_V0_periodic_cube_plane_wave_modes_filter_to_scalar_multiple():
    """Same mesh: every eigenvector of the discrete Laplacian is filtered to a scalar multiple of itself, and
    the lowest non-zero eigenvalue is 1/2 (2 pi / L)^2 to spectral accuracy (6-fold degenerate)."""
    wl = make_workload(None, n=3, p=3, L=6.0, atoms_per_side=0, n_gaussians=0, nonlocal_=False, smooth_field=0.0,
                       seed_base=3)
    op = orc.operator_from_workload(wl)
    H = orc.apply_H(op, np.eye(op.n_dofs))
    lam, V = np.linalg.eigh(0.5 * (H + H.T))
    assert abs(lam[0]) < 1e-10 and np.allclose(lam[1:7], 0.5 * (2 * np.pi / 6.0) ** 2, rtol=1e-3)   # p=3: ~3e-4; spectral convergence is pinned in test_oracle_operator.py
    a0, a, b, m = -0.1, 2.0, lam[-1] * 1.01, 12
    e, c = (b - a) / 2, (b + a) / 2
    Y = orc.chebyshev_filter(op, V[:, :40], m, a, b, a0)
    gain = cheb_T(m, (lam[:40] - c) / e) / cheb_T(m, np.array([(a0 - c) / e]))[0]
    assert np.allclose(Y, V[:, :40] * gain[None, :], atol=1e-11 * np.max(np.abs(gain)))


def test_filter_linearity_column_independence_and_chunking(tiny_eig):
    op, lam, _ = tiny_eig
    a0, a, b, m = lam[0], lam[0] + 2.0, lam[-1] + 0.1, 7
    X = random_block(op.n_dofs, range(10), 9)
    Y = orc.chebyshev_filter(op, X, m, a, b, a0)
    Yc = np.concatenate([orc.chebyshev_filter(op, X[:, j0:j0 + 4], m, a, b, a0) for j0 in (0, 4, 8)], axis=1)
    assert np.array_equal(Y.shape, Yc.shape) and np.allclose(Y, Yc, rtol=1e-13, atol=1e-13 * np.abs(Y).max())
    w = np.array([0.3, -1.7, 2.2])
    Yl = orc.chebyshev_filter(op, X[:, :3] @ w[:, None], m, a, b, a0)
    assert np.allclose(Yl[:, 0], Y[:, :3] @ w, rtol=1e-12, atol=1e-12 * np.abs(Y).max())


def test_filter_argument_errors(tiny_eig):
    op, lam, _ = tiny_eig
    X = np.ones((op.n_dofs, 1))
    with pytest.raises(ValueError):
        orc.chebyshev_filter(op, X, 0, 1.0, 2.0, 0.0)
    with pytest.raises(ValueError):
        orc.chebyshev_filter(op, X, 3, 2.0, 1.0, 0.0)
    with pytest.raises(ValueError):
        orc.chebyshev_filter(op, X, 3, 1.0, 2.0, 1.5)


def test_lanczos_bound_and_rayleigh_ritz_against_dense_eigh(tiny_eig):
    op, lam, V = tiny_eig
    v0 = np.random.default_rng(1).standard_normal(op.n_dofs)
    b, lmin = orc.lanczos_upper_bound(op, v0, 20)
    assert b >= lam[-1] and b <= lam[-1] + 0.5 * (lam[-1] - lam[0])
    assert lam[0] <= lmin <= lam[-1]                               # Ritz values lie inside the spectrum
    # Rayleigh-Ritz on an invariant subspace returns its eigenvalues exactly, whatever the basis of the subspace
    R = np.random.default_rng(2).standard_normal((6, 6))
    theta = orc.rayleigh_ritz(op, V[:, 2:8] @ R)
    assert np.allclose(theta, lam[2:8], rtol=0, atol=1e-10)
    Y = V[:, 2:8] @ R
    theta2 = orc.ritz_values_of_block(Y, orc.apply_H(op, Y))
    assert np.allclose(theta2, lam[2:8], rtol=0, atol=1e-10)
    # Cauchy interlacing for an arbitrary subspace
    Q, _ = np.linalg.qr(np.random.default_rng(3).standard_normal((op.n_dofs, 5)))
    th = orc.rayleigh_ritz(op, Q)
    assert np.all(th >= lam[:5] - 1e-10) and np.all(th <= lam[-5:] + 1e-10)


def test_projection_matrices_closed_forms_on_eigenvectors(tiny_eig):
    """Algorithm 2 step 1: on orthonormal eigenvectors S = I and H^ = diag(lambda); for a
    mixture Y = V R of eigenvectors S = R^T R and H^ = R^T diag(lambda) R; S and H^ are symmetric; and the generalised
    eigenvalues of (H^, S) are the eigenvalues of the invariant subspace (LAPACK via scipy)."""
    import scipy.linalg
    op, lam, V = tiny_eig
    S, Hh = orc.projection_matrices(op, V[:, 3:10])
    assert np.allclose(S, np.eye(7), atol=1e-12) and np.allclose(Hh, np.diag(lam[3:10]), atol=1e-10)
    R = np.random.default_rng(8).standard_normal((7, 7))
    S, Hh = orc.projection_matrices(op, V[:, 3:10] @ R)
    assert np.allclose(S, R.T @ R, atol=1e-11)
    assert np.allclose(Hh, R.T @ np.diag(lam[3:10]) @ R, atol=1e-9)
    assert np.allclose(S, S.T, atol=1e-12) and np.allclose(Hh, Hh.T, atol=1e-10)
    theta = scipy.linalg.eigh(0.5 * (Hh + Hh.T), S, eigvals_only=True)
    assert np.allclose(theta, lam[3:10], atol=1e-9)


def test_config1_stored_bounds_follow_the_recipe_and_bound_the_spectrum():
    """bounds.json (written by oracle/make_bounds.py) for config 1: b >= lambda_max and a0 <= a < b against a
    dense eigh of the 4096-dof operator, and both recipes reproduce from their seeds."""
    spec = CONFIGS[1]
    wl = make_workload(1)
    op = orc.operator_from_workload(wl)
    H = orc.apply_H(op, np.eye(op.n_dofs))
    assert np.abs(H - H.T).max() <= 1e-12 * np.abs(H).max()
    lam = np.linalg.eigvalsh(0.5 * (H + H.T))
    for recipe in ("A", "B"):
        a0, a, b = load_bounds("1", recipe)
        assert b >= lam[-1] and a0 <= a < b and a0 >= lam[0] - 1e-9
    v0 = np.random.default_rng(spec.seed_base + SEED_LANCZOS).standard_normal(wl.n_dofs)
    b, lmin = orc.lanczos_upper_bound(op, v0, 20)
    Q, _ = np.linalg.qr(np.random.default_rng(spec.seed_base + SEED_RR).standard_normal((wl.n_dofs, 30)))
    th = orc.rayleigh_ritz(op, Q)
    a0A, aA, bA = load_bounds("1", "A")
    assert np.isclose(b, bA, rtol=1e-10) and np.isclose(th[0], a0A, rtol=1e-9) and np.isclose(th[-1], aA, rtol=1e-9)
    a0B, aB, bB = load_bounds("1", "B")
    assert np.isclose(lmin, a0B, rtol=1e-9)


def test_bounds_table_is_complete_and_ordered():
    path = os.path.join(os.path.dirname(os.path.dirname(os.path.abspath(__file__))), "workloads", "bounds.json")
    with open(path) as f:
        table = json.load(f)
    for spec in CONFIGS.values():
        for recipe in ("A", "B"):
            e = table[spec.bounds_key][recipe]
            assert e["a0"] <= e["a"] < e["b"]


@pytest.mark.parametrize("jitter", [0.0, 0.12])
def test_apply_H_rows_equals_rows_of_apply_H(jitter):
    wl = make_workload(None, n=3, p=2, L=6.0, mesh_jitter=jitter, atoms_per_side=1, n_gaussians=0, nonlocal_=True,
                       smooth_field=0.05, seed_base=21, r_cut=2.2)
    assert wl.n_proj == 8 and wl.proj_cell_ptr[-1] > 8
    op = orc.operator_from_workload(wl)
    X = random_block(op.n_dofs, range(4), 3)
    rows = [0, 5, 17, 100, op.n_dofs - 1]                        # vertex, edge, face and interior dofs
    Y = orc.apply_H(op, X)
    Yr = orc.apply_H_rows(wl, op.M, X, rows)
    assert np.allclose(Yr, Y[rows], rtol=1e-12, atol=1e-13 * np.abs(Y).max())


# ------------------------------------------------------------------------------------------------------------
# Rayleigh-Ritz step of Algorithm 2 with the paper's mixed-precision blocking
# ------------------------------------------------------------------------------------------------------------
def test_cholesky_inverse_against_lapack_and_definition():
    rng = np.random.default_rng(11)
    for n in (1, 2, 7, 40):
        A = rng.standard_normal((n + 5, n))
        S = A.T @ A + 0.1 * np.eye(n)
        L, Linv = orc.cholesky_inverse(S)
        assert np.allclose(L, np.linalg.cholesky(S), rtol=1e-12, atol=1e-13)      # library routine
        assert np.allclose(np.triu(L, 1), 0) and np.all(np.diag(L) > 0)
        assert np.allclose(L @ L.T, S, rtol=1e-12, atol=1e-12)                    # definition
        assert np.allclose(Linv @ L, np.eye(n), atol=1e-11) and np.allclose(np.triu(Linv, 1), 0)
    with pytest.raises(np.linalg.LinAlgError):
        orc.cholesky_inverse(np.array([[1.0, 2.0], [2.0, 1.0]]))


def test_mixed_precision_overlap_blocks():
    """Diagonal blocks are the FP64 product bit for bit, off-diagonal blocks carry an FP32-sized error that scales with
    the column norms (and vanishes with the off-diagonal content: orthonormal input gives the identity to FP32
    rounding of exact zeros); block = N reduces to the FP64 overlap; a transposed / wrong-block implementation fails."""
    rng = np.random.default_rng(12)
    n, N, blk = 600, 24, 8
    Y = rng.standard_normal((n, N)) * np.logspace(0, 2, N)[None, :]
    S64 = Y.T @ Y
    Sm = orc.overlap_mixed(Y, blk)
    nrm = np.linalg.norm(Y, axis=0)
    for j0 in range(0, N, blk):
        assert np.array_equal(Sm[j0:j0 + blk, j0:j0 + blk], S64[j0:j0 + blk, j0:j0 + blk])
    off = np.ones((N, N), dtype=bool)
    for j0 in range(0, N, blk):
        off[j0:j0 + blk, j0:j0 + blk] = False
    err = np.abs(Sm - S64) / np.outer(nrm, nrm)
    assert 1e-10 < err[off].max() <= 20 * np.finfo(np.float32).eps      # FP32-sized, not FP64-sized
    assert np.array_equal(orc.overlap_mixed(Y, N), S64)
    Q, _ = np.linalg.qr(rng.standard_normal((n, N)))
    Sq = orc.overlap_mixed(Q, blk)
    assert np.max(np.abs(Sq - np.eye(N))) <= 5e-7 and np.max(np.abs(np.diag(Sq) - 1)) <= 1e-14


def test_mixed_precision_projected_hamiltonian_blocks_and_ritz_values():
    """Eq. 39: only the fr-fr block is FP64 (bit-equal to the FP64 product), the other three are FP32 products; for a
    nearly converged subspace (H^ nearly diagonal) the n_fr highest Ritz values of the mixed matrices agree with the
    FP64 ones far below the FP32 level -- the property the paper's blocking rests on."""
    wl = make_workload(None, n=3, p=3, L=6.0, atoms_per_side=1, n_gaussians=0, nonlocal_=True, smooth_field=0.05,
                       seed_base=61)
    op = orc.operator_from_workload(wl)
    rng = np.random.default_rng(13)
    N, n_oc = 16, 10
    Y = rng.standard_normal((wl.n_dofs, N))
    HY = orc.apply_H(op, Y)
    Hm = orc.projected_hamiltonian_mixed(Y, HY, n_oc)
    H64 = Y.T @ HY
    assert np.array_equal(Hm[n_oc:, n_oc:], H64[n_oc:, n_oc:])
    assert not np.array_equal(Hm[:n_oc, :n_oc], H64[:n_oc, :n_oc]) and not np.array_equal(Hm[n_oc:, :n_oc], H64[n_oc:, :n_oc])
    assert np.max(np.abs(Hm - H64)) <= 1e-5 * np.max(np.abs(H64))
    # nearly converged subspace: a few filter + orthonormalisation passes
    b, lmin = orc.lanczos_upper_bound(op, rng.standard_normal(wl.n_dofs), 20)
    for _ in range(8):
        th = orc.ritz_values_of_block(Y, orc.apply_H(op, Y))
        Y, _ = np.linalg.qr(orc.chebyshev_filter(op, Y, 12, float(th[-1]), b, float(th[0]) - 1e-3))
    Y = Y * (1.0 + 0.2 * rng.standard_normal(N))[None, :]         # not normalised: S is diagonal-dominant, not the identity
    HY = orc.apply_H(op, Y)
    n_fr = N - n_oc
    d64, _, _ = orc.rayleigh_ritz_gep(Y.T @ Y, Y.T @ HY, n_fr)
    dm, _, _ = orc.rayleigh_ritz_gep(orc.overlap_mixed(Y, 4), orc.projected_hamiltonian_mixed(Y, HY, n_oc), n_fr)
    conv = np.abs(d64 - orc.ritz_values_of_block(Y, HY)[-n_fr:])
    assert np.max(conv) <= 1e-9                                    # the GEP route equals the Rayleigh-Ritz measure
    assert np.max(np.abs(dm[:3] - d64[:3])) <= 1e-7, np.abs(dm - d64)


def test_rayleigh_ritz_gep_and_mixed_orthonormal_basis():
    """Algorithm 2 steps 2-3 on an invariant subspace written in a random basis: D_fr are the top eigenvalues, Psi^R =
    Y Q_fr are eigenvectors, Psi^o = Y L^-T is orthonormal; the mixed SP/DP form of Psi^o differs by an FP32-sized term
    that vanishes when L^-T is diagonal (orthogonal input columns)."""
    rng = np.random.default_rng(14)
    n, N, n_fr = 60, 9, 4
    A = rng.standard_normal((n, n))
    H = 0.5 * (A + A.T)
    ev, V = np.linalg.eigh(H)
    Y = V[:, :N] @ rng.standard_normal((N, N))
    D, Q, Linv = orc.rayleigh_ritz_gep(Y.T @ Y, Y.T @ (H @ Y), n_fr)
    assert np.allclose(D, ev[N - n_fr:N], atol=1e-9)
    R = Y @ Q
    assert np.allclose(H @ R, R * D[None, :], atol=1e-8)
    Po = Y @ Linv.T
    assert np.allclose(Po.T @ Po, np.eye(N), atol=1e-9)
    Pm = orc.orthonormal_basis_mixed(Y, Linv.T)
    assert 0 < np.max(np.abs(Pm - Po)) <= 1e-4 * np.max(np.abs(Po))
    Yo = V[:, :N] * (1.0 + rng.random(N))[None, :]                 # orthogonal columns: L^-T is diagonal
    _, _, Li = orc.rayleigh_ritz_gep(Yo.T @ Yo, Yo.T @ (H @ Yo), n_fr)
    Li_d = np.diag(np.diag(Li))
    assert np.allclose(orc.orthonormal_basis_mixed(Yo, Li_d.T), Yo @ Li_d.T, rtol=1e-15, atol=0)
