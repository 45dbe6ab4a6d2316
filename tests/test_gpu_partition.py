"""Cell-partitioned operation on ONE GPU, `-m gpu`: R host threads play the ranks of paper_2203_07820_b200/partition.py on
the same device (each with its own part operator; the all-reduce is a host barrier + a device sum, so no kernel ever waits
for another one), and the assembled result is compared with the ORACLE on the whole mesh at the FP64 tolerances
(<= 1e-10; FP32 boundary payload: <= 1e-5).  NCCL itself is not exercised here (one GPU); the gloo test in
test_partition_cpu.py covers the torch.distributed path of the same communicator interface."""
import threading

import numpy as np
import pytest

pytestmark = pytest.mark.gpu


class ThreadComm:
    """all_reduce over R threads of one process: deposit, barrier, rank 0 sums on the device and copies back, barrier."""

    class World:
        def __init__(self, n):
            self.n, self.barrier, self.slots = n, threading.Barrier(n), [None] * n

    class _Done:
        def wait(self):
            return None

    def __init__(self, world_obj, rank):
        self.w, self.rank, self.world = world_obj, rank, world_obj.n

    def all_reduce(self, t, async_op=False):
        import torch
        w = self.w
        w.slots[self.rank] = t
        w.barrier.wait()
        if self.rank == 0:
            total = w.slots[0].clone()
            for s in w.slots[1:]:
                total += s
            for s in w.slots:
                s.copy_(total)
            torch.cuda.synchronize()
        w.barrier.wait()
        return ThreadComm._Done() if async_op else None

    def all_reduce_host(self, a):
        w = self.w
        w.slots[self.rank] = a
        w.barrier.wait()
        total = sum(w.slots[1:], w.slots[0].copy())
        w.barrier.wait()
        return total


def run_ranks(world, fn):
    """fn(comm) on `world` threads; returns the list of results, re-raises the first exception."""
    w = ThreadComm.World(world)
    out, err = [None] * world, [None] * world

    def main(r):
        try:
            import torch
            torch.cuda.set_device(0)
            out[r] = fn(ThreadComm(w, r))
        except BaseException as e:          # noqa: BLE001
            err[r] = e
            w.barrier.abort()

    ts = [threading.Thread(target=main, args=(r,)) for r in range(world)]
    for t in ts:
        t.start()
    for t in ts:
        t.join()
    for e in err:
        if e is not None and not isinstance(e, threading.BrokenBarrierError):
            raise e
    for e in err:
        if e is not None:
            raise e
    return out


def workload(p=4, n=4, atoms_per_side=2):
    from workloads.generate import make_workload
    return make_workload(None, n=n, p=p, L=2.0 * n, mesh_jitter=0.1, atoms_per_side=atoms_per_side, n_gaussians=0, nonlocal_=True,
                         smooth_field=0.05, seed_base=56, r_cut=2.2)


# aps = atoms per side.  With one atom every cell has at most 8 projectors, the parts run the sum-factorised kernel and the
# filter goes through the accumulate-only exchange (asserted); with 2^3 atoms some cells see more than 16 projectors, the
# parts run the dense kernel and the filter takes H~X + exchange + recurrence pass.
@pytest.mark.parametrize("world,p,fp32,aps", [(2, 4, False, 2), (3, 6, False, 2), (4, 3, False, 2), (2, 6, True, 2),
                                              (2, 6, False, 1), (3, 4, True, 1), (4, 5, False, 1)])
def test_partitioned_apply_and_filter_match_the_oracle_on_the_whole_mesh(world, p, fp32, aps):
    import torch
    from oracle import chfsi_oracle as orc
    from paper_2203_07820_b200.partition import CellPartition, PartitionedOperator
    from workloads.generate import random_block
    wl = workload(p=p, n=4 if p <= 4 else 3, atoms_per_side=aps)
    oop = orc.operator_from_workload(wl)
    B, m = 24, 6
    X = random_block(wl.n_dofs, range(B), 9)
    bnd, lmin = orc.lanczos_upper_bound(oop, np.random.default_rng(5).standard_normal(wl.n_dofs), 20)
    a0, a, b = lmin, lmin + 0.1 * (bnd - lmin), bnd
    Yo = orc.apply_H(oop, X)
    Fo = orc.chebyshev_filter(oop, X, m, a, b, a0)
    cp = CellPartition(wl, world)
    assert len(cp.shared_dofs) > 0
    # atoms whose support straddles a partition face: the projector all-reduce is really needed
    owners = [set(int(cp.owner[int(c)]) for c in wl.proj_cell_idx[int(wl.proj_cell_ptr[j]):int(wl.proj_cell_ptr[j + 1])])
              for j in range(wl.n_proj)]
    assert any(len(o) > 1 for o in owners)

    def rank_main(comm):
        part = PartitionedOperator(wl, comm=comm, partition=cp, boundary_fp32=fp32)
        Xl = part.scatter_block(X)
        Y = part.apply_H(Xl)
        F = Xl.clone()
        part.chebyshev_filter_chunked(F, 8, m, a, b, a0)            # three chunks: a pair in flight, then a single one
        if aps == 1:
            assert part.op.accumulate_supported(F[:, :8], Xl[:, :8])     # ... in scaled blocks (the cell kernel accumulates)
        F3 = Xl.clone()
        part.chebyshev_filter_chunked(F3, 8, m, a, b, a0, scaled=False)   # H~X, exchange, separate recurrence pass
        err3 = float((F3 - F).norm() / F.norm())
        assert err3 <= (1e-5 if fp32 else 1e-12), err3
        torch.cuda.synchronize()
        res = (part.part.dofs, Y.cpu().numpy(), F.cpu().numpy(), part.op.launch_count())
        part.close()
        return res

    res = run_ranks(world, rank_main)
    tol = 1e-5 if fp32 else 1e-10
    Yg, Fg, seen = np.zeros_like(Yo), np.zeros_like(Fo), np.zeros(wl.n_dofs, dtype=int)
    for dofs, Y, F, launches in res:
        assert launches > 0
        # replicas of shared rows agree bit for bit between the ranks that hold them
        both = seen[dofs] > 0
        assert np.array_equal(Yg[dofs[both]], Y[both]) and np.array_equal(Fg[dofs[both]], F[both])
        Yg[dofs], Fg[dofs] = Y, F
        seen[dofs] += 1
    assert seen.min() >= 1
    for got, want, what in ((Yg, Yo, "apply_H"), (Fg, Fo, f"filter m={m}")):
        err = float(np.linalg.norm(got - want) / np.linalg.norm(want))
        emax = float(np.max(np.abs(got - want)) / np.max(np.abs(want)))
        assert err <= tol and emax <= tol, f"world {world} {what}: rel Frobenius {err:.3e}, max-norm {emax:.3e}"


@pytest.mark.parametrize("aps", [1, 2])
def test_single_part_equals_the_plain_operator(aps):
    """world = 1: the phased application (coefficients, then H~X with given coefficients) is the plain chfsi_apply_H, and the
    filter (aps = 1: through the accumulate-only path, like chfsi_chebyshev_filter itself) is the plain filter."""
    import torch
    from paper_2203_07820_b200 import Operator
    from paper_2203_07820_b200.partition import PartitionedOperator
    from workloads.generate import random_block
    wl = workload(p=6, n=3, atoms_per_side=aps)
    part = PartitionedOperator(wl)
    op = Operator.from_workload(wl)
    assert np.allclose(part.mass, op.mass_diag().cpu().numpy(), rtol=1e-14, atol=0)
    X = torch.tensor(random_block(wl.n_dofs, range(16), 2), device="cuda")
    assert torch.equal(part.apply_H(X), op.apply_H(X))
    F1, F2 = X.clone(), X.clone()
    part.chebyshev_filter(F1, 5, 0.5, 300.0, 0.1)
    op.chebyshev_filter(F2, 5, 0.5, 300.0, 0.1)
    assert float((F1 - F2).norm() / F2.norm()) <= 1e-13
    F3, F4 = X.clone(), X.clone()                                   # even degree: the final rescale is in place
    part.chebyshev_filter(F3, 6, 0.5, 300.0, 0.1)
    op.chebyshev_filter(F4, 6, 0.5, 300.0, 0.1)
    assert float((F3 - F4).norm() / F4.norm()) <= 1e-13
    part.close(); op.close()


_NCCL_WORLD1 = r"""
import os, sys
import torch, torch.distributed as dist
torch.cuda.set_device(0)
dist.init_process_group("nccl", rank=0, world_size=1, device_id=torch.device("cuda", 0))
from paper_2203_07820_b200 import Operator
from paper_2203_07820_b200.partition import PartitionedOperator, TorchComm
from workloads.generate import make_workload, random_block
wl = make_workload(None, n=3, p=6, L=6.0, mesh_jitter=0.1, atoms_per_side=1, n_gaussians=0, nonlocal_=True, smooth_field=0.05,
                   seed_base=56, r_cut=2.2)
part = PartitionedOperator(wl, comm=TorchComm())
op = Operator.from_workload(wl)
X = torch.tensor(random_block(wl.n_dofs, range(32), 2), device="cuda")
assert torch.equal(part.apply_H(X), op.apply_H(X))
F1, F2, F3 = X.clone(), X.clone(), X.clone()
part.chebyshev_filter_chunked(F1, 8, 7, 0.5, 300.0, 0.1)                  # async all-reduces, two chunks in flight
op.chebyshev_filter(F2, 7, 0.5, 300.0, 0.1)
part.chebyshev_filter_chunked(F3, 8, 7, 0.5, 300.0, 0.1, scaled=False)
torch.cuda.synchronize()
assert float((F1 - F2).norm() / F2.norm()) <= 1e-13 and float((F3 - F2).norm() / F2.norm()) <= 1e-13
dist.destroy_process_group()
print("NCCL-WORLD1-OK")
"""


def test_torch_distributed_communicator_over_nccl_with_one_rank():
    """TorchComm on the NCCL backend (the communicator `bench.py --gpus N --partition` uses), world size 1, in a process of its
    own: process-group set-up with a device id, the host all-reduce of the mass through a device tensor, synchronous and
    asynchronous device all-reduces ordered against the library's kernels on torch's current stream.  More ranks need more GPUs."""
    import os
    import subprocess
    import sys
    env = dict(os.environ, MASTER_ADDR="127.0.0.1", MASTER_PORT=str(29600 + os.getpid() % 300), RANK="0", WORLD_SIZE="1")
    root = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
    r = subprocess.run([sys.executable, "-c", _NCCL_WORLD1], cwd=root, env=env, capture_output=True, text=True, timeout=600)
    assert r.returncode == 0 and "NCCL-WORLD1-OK" in r.stdout, r.stdout[-2000:] + r.stderr[-4000:]
