"""Host logic of the cell-partitioned (multi-GPU) form (paper_2203_07820_b200/partition.py),
`-m "not gpu"`: the partition bookkeeping, the mass of the whole mesh assembled from the parts over a world-size-2 gloo
group, and the algebra of the boundary sum (parts' contributions on shared dofs add up to H~ X of the whole mesh) with the
ORACLE standing in for the part operators."""
import multiprocessing as mp
import os

import numpy as np
import pytest

from workloads.generate import make_workload


def small_workload(nonlocal_=True, n=4, p=2, jitter=0.1):
    return make_workload(None, n=n, p=p, L=2.0 * n, mesh_jitter=jitter, atoms_per_side=2, n_gaussians=0, nonlocal_=nonlocal_,
                         smooth_field=0.05, seed_base=55, r_cut=2.2)


@pytest.mark.parametrize("world", [1, 2, 3, 4])
def test_partition_covers_the_mesh_and_maps_back(world):
    from paper_2203_07820_b200.partition import CellPartition
    wl = small_workload()
    cp = CellPartition(wl, world)
    cd = np.asarray(wl.cell_dofs)
    counts = np.bincount(cp.owner, minlength=world)
    assert counts.sum() == cd.shape[0] and counts.min() >= cd.shape[0] // world           # balanced, every cell once
    touched = np.zeros(wl.n_dofs, dtype=int)
    n_q = wl.veff_q.shape[1]
    proj_cells_seen = 0
    for r in range(world):
        lp = cp.local(r)
        assert np.array_equal(lp.dofs[lp.cell_dofs], cd[lp.cells])                          # local ids map back
        assert np.array_equal(lp.cell_vertices.reshape(-1, 24), np.asarray(wl.cell_vertices).reshape(-1, 24)[lp.cells])
        touched[lp.dofs] += 1
        assert np.array_equal(lp.dofs[lp.shared_rows], cp.shared_dofs[lp.shared_slots])     # rows <-> slots of shared dofs
        assert lp.shared_owner.dtype == np.uint8 and lp.shared_owner.shape == lp.shared_rows.shape
        # projectors: the local CSR is the global one restricted to this rank's cells, samples and couplings carried along
        for jl, j in enumerate(lp.proj_ids):
            assert lp.D[jl] == wl.D[j]
            glob = {int(wl.proj_cell_idx[k]): k for k in range(int(wl.proj_cell_ptr[j]), int(wl.proj_cell_ptr[j + 1]))}
            for kl in range(int(lp.proj_cell_ptr[jl]), int(lp.proj_cell_ptr[jl + 1])):
                gc = int(lp.cells[lp.proj_cell_idx[kl]])
                assert gc in glob and np.array_equal(lp.chi_q[kl], wl.chi_q[glob[gc]])
                proj_cells_seen += 1
        assert lp.chi_q.shape == (len(lp.proj_cell_idx), n_q)
    assert touched.min() >= 1
    assert np.array_equal(np.nonzero(touched >= 2)[0], cp.shared_dofs)
    owners = np.zeros(len(cp.shared_dofs), dtype=int)                                       # every shared dof has ONE owner
    for r in range(world):
        lp = cp.local(r)
        np.add.at(owners, lp.shared_slots, lp.shared_owner)
    assert np.all(owners == 1)
    assert proj_cells_seen == len(wl.proj_cell_idx)                                         # every (projector, cell) pair once
    if world == 1:
        assert len(cp.shared_dofs) == 0


def test_scaled_scalars_reproduce_the_three_term_recurrence():
    """W_k = s_k Y_k with W_k = W_{k-2} + g_k (H~ - c) W_{k-1} (U14) on scalars: for an eigenvalue lam the classic
    recurrence gives y_m, the scaled one w_m / s_m: equal; and the guard returns None when s_k leaves the FP32 range."""
    from paper_2203_07820_b200.partition import PartitionedOperator as PO
    m, a, b, a0 = 12, 0.4, 30.0, -0.3
    scal, c = PO.recurrence_scalars(m, a, b, a0)
    gam, inv_sm, c2 = PO.scaled_scalars(m, a, b, a0)
    assert c2 == c and len(gam) == m
    for lam in (-0.3, 0.1, 5.0, 29.0):
        y0, y1 = 1.0, scal[0][0] * (lam - c)
        w0, w1 = 1.0, gam[0] * (lam - c)
        for k in range(1, m):
            y0, y1 = y1, scal[k][0] * (lam - c) * y1 - scal[k][1] * y0
            w0, w1 = w1, w0 + gam[k] * (lam - c) * w1
        assert abs(w1 * inv_sm - y1) <= 1e-12 * max(1.0, abs(y1))
    assert PO.scaled_scalars(60, 0.4, 30.0, -30.0, precision=32) is None and PO.scaled_scalars(60, 0.4, 30.0, -30.0) is not None


def test_delta_exchange_with_owner_correction_sums_to_the_whole_mesh_update():
    """The accumulate-only exchange (include/chfsi.h: chfsi_pack_rows_delta / chfsi_unpack_rows_sum) with the ORACLE as the part
    operators: every part adds g (H~_part - c) X to its copy of W, subtracting c X once per dof it holds; what travels is
    W_new - W_old on the shared rows, with g c X put back by the parts that do not own the dof; base + sum = W + g (H~ - c) X."""
    from oracle import chfsi_oracle as orc
    from paper_2203_07820_b200 import mesh_mass
    from paper_2203_07820_b200.partition import CellPartition
    wl = small_workload(nonlocal_=False)
    world, g, c = 3, -0.37, 1.9
    cp = CellPartition(wl, world)
    Mg = mesh_mass(wl.p, wl.cell_dofs, wl.cell_vertices, wl.n_dofs)
    rng = np.random.default_rng(8)
    X, W = rng.standard_normal((wl.n_dofs, 4)), rng.standard_normal((wl.n_dofs, 4))
    want = W + g * (orc.apply_H(orc.operator_from_workload(wl), X) - c * X)
    buf = np.zeros((len(cp.shared_dofs), 4))
    locals_ = []
    for r in range(world):
        lp = cp.local(r)
        oop = orc.build_operator(wl.p, lp.cell_dofs, lp.cell_vertices, len(lp.dofs), lp.veff_q)
        oop.M = Mg[lp.dofs]
        Wl = W[lp.dofs] + g * (orc.apply_H(oop, X[lp.dofs]) - c * X[lp.dofs])               # what the part's kernel leaves
        base = W[lp.dofs][lp.shared_rows]
        buf[lp.shared_slots] += Wl[lp.shared_rows] - base + g * c * X[lp.dofs][lp.shared_rows] * (1 - lp.shared_owner)[:, None]
        locals_.append((lp, Wl, base))
    for lp, Wl, base in locals_:
        Wl[lp.shared_rows] = base + buf[lp.shared_slots]
        assert np.max(np.abs(Wl - want[lp.dofs])) <= 1e-12 * np.max(np.abs(want))


def test_mesh_mass_of_the_library_equals_the_oracle_and_the_volume():
    from oracle import chfsi_oracle as orc
    from paper_2203_07820_b200 import mesh_mass
    wl = small_workload(p=3)
    M = mesh_mass(wl.p, wl.cell_dofs, wl.cell_vertices, wl.n_dofs)
    assert np.allclose(M, orc.mass_diagonal(wl.p, wl.cell_dofs, wl.cell_vertices, wl.n_dofs), rtol=1e-13, atol=0)
    assert abs(M.sum() - 8.0 ** 3) <= 1e-10 * 8.0 ** 3                                      # sum M = volume of the periodic box


def _rank_main(rank, world, port, q):
    """One gloo rank: mass of the whole mesh at its dofs, and its (oracle) contribution to H~ X with the boundary sum."""
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    import torch
    import torch.distributed as dist
    from oracle import chfsi_oracle as orc
    from paper_2203_07820_b200.partition import CellPartition, TorchComm, global_mass_at
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        wl = small_workload(nonlocal_=False)
        comm = TorchComm()
        cp = CellPartition(wl, world)
        lp = cp.local(rank)
        mass = global_mass_at(lp, cp, wl.p, comm)
        # the part as an oracle operator with the mass of the whole mesh; its apply_H is the part's contribution
        oop = orc.build_operator(wl.p, lp.cell_dofs, lp.cell_vertices, len(lp.dofs), lp.veff_q)
        oop.M = mass
        X = np.random.default_rng(3).standard_normal((wl.n_dofs, 5))
        Y = orc.apply_H(oop, X[lp.dofs])
        buf = torch.zeros((len(cp.shared_dofs), 5), dtype=torch.float64)
        buf[torch.from_numpy(lp.shared_slots.astype(np.int64))] = torch.from_numpy(Y[lp.shared_rows])
        comm.all_reduce(buf)
        Y[lp.shared_rows] = buf.numpy()[lp.shared_slots]
        q.put((rank, lp.dofs, mass, Y))
    finally:
        dist.destroy_process_group()


def test_world_size_2_gloo_mass_and_boundary_sum_reproduce_the_whole_mesh():
    from oracle import chfsi_oracle as orc
    from paper_2203_07820_b200 import mesh_mass
    world, port = 2, 29500 + os.getpid() % 2000
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    procs = [ctx.Process(target=_rank_main, args=(r, world, port, q)) for r in range(world)]
    for p in procs:
        p.start()
    res = [q.get(timeout=240) for _ in range(world)]
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    wl = small_workload(nonlocal_=False)
    Mg = mesh_mass(wl.p, wl.cell_dofs, wl.cell_vertices, wl.n_dofs)
    X = np.random.default_rng(3).standard_normal((wl.n_dofs, 5))
    Yg = orc.apply_H(orc.operator_from_workload(wl), X)
    for rank, dofs, mass, Y in res:
        assert np.allclose(mass, Mg[dofs], rtol=1e-14, atol=0)
        assert np.max(np.abs(Y - Yg[dofs])) <= 1e-12 * np.max(np.abs(Yg))


def test_part_entry_points_report_argument_errors_without_a_device():
    import ctypes as C
    from paper_2203_07820_b200 import load_library
    from paper_2203_07820_b200.binding import _KPoint, _Mesh, _Potential
    lib = load_library()
    M = np.zeros(8)
    assert lib.chfsi_mesh_mass(None, M.ctypes.data) == -1
    cd = np.arange(8, dtype=np.int32).reshape(1, 8)
    cv = np.zeros((1, 8, 3))                                                 # degenerate cell: non-positive Jacobian
    mesh = _Mesh(1, 1, 8, cd.ctypes.data, cv.ctypes.data)
    assert lib.chfsi_mesh_mass(C.byref(mesh), M.ctypes.data) == -2
    assert b"Jacobian" in lib.chfsi_last_error(None)
    mesh9 = _Mesh(9, 1, 8, cd.ctypes.data, cv.ctypes.data)
    assert lib.chfsi_mesh_mass(C.byref(mesh9), M.ctypes.data) == -5
    h = C.c_void_p()
    vq = np.zeros((1, 27))
    pot = _Potential(vq.ctypes.data)
    assert lib.chfsi_create_part(C.byref(h), C.byref(mesh), C.byref(pot), None, None, 64, 0, None) == -1     # dof_mass == NULL
    assert lib.chfsi_create_k(C.byref(h), C.byref(mesh), C.byref(pot), None, None, 0, None) == -1           # kpoint == NULL
    kp = _KPoint()
    kp.k[0], kp.k[1], kp.k[2] = float("nan"), 0.0, 0.0
    assert lib.chfsi_create_k(C.byref(h), C.byref(mesh), C.byref(pot), None, C.byref(kp), 0, None) == -1    # non-finite k
    mesh7 = _Mesh(7, 1, 512, cd.ctypes.data, cv.ctypes.data)
    kp.k[0] = 0.1
    assert lib.chfsi_create_k(C.byref(h), C.byref(mesh7), C.byref(pot), None, C.byref(kp), 0, None) == -5   # p = 7
    assert h.value is None
    for fn, args in ((lib.chfsi_projector_coefficients, (None, None, 0, 0, None, None, None)),
                     (lib.chfsi_apply_H_with_coefficients, (None, None, 0, None, 0, 0, None, None, None)),
                     (lib.chfsi_pack_rows, (None, None, 0, 0, None, None, 0, None, 64, None)),
                     (lib.chfsi_unpack_rows, (None, None, 64, None, None, 0, None, 0, 0, None)),
                     (lib.chfsi_recurrence_update, (None, None, 0, None, 0, None, 0, 0, 1.0, 0.0, 0.0, None)),
                     (lib.chfsi_accumulate_supported, (None, None, 0, None, 0, 0, None, None)),
                     (lib.chfsi_apply_shifted_with_coefficients, (None, None, 0, None, 0, 0, 1.0, 0.0, 1, None, None, None)),
                     (lib.chfsi_pack_rows_delta, (None, None, 0, None, None, 0, None, 0.0, 0, None, None, 0, None, 64, None)),
                     (lib.chfsi_unpack_rows_sum, (None, None, 64, None, None, None, 0, None, 0, 0, None))):
        assert fn(*args) == -1
