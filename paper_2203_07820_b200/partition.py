"""Cell-partitioned (multi-GPU) form of H~ X and of the Chebyshev filter: the paper's domain decomposition over MPI tasks
/ GPUs, with one sum of the rows of the shared dofs per H~ application, all vectors of a block in one
message, optionally in FP32, and the projector coefficients summed over the parts (Alg. 4 step 3,
PAPER.md:526).

One process per GPU.  Every rank holds the description of the whole mesh on the host (connectivity, vertices, samples),
builds the SAME `CellPartition` from it, creates an operator on its own cells (chfsi_create_part) and keeps the rows of
the dofs its cells touch; rows of shared dofs are replicated on the ranks that share them and kept identical.

    H~ X:   P_part = D C_part^T X          ->  all-reduce over the ranks (n_proj x B, small)
            Y      = part's contribution   ->  rows of the shared dofs: pack, all-reduce, unpack (FP64 or FP32 payload)
    filter: Y_k = alpha_k (H~ Y_{k-1} - c Y_{k-1}) - beta_k Y_{k-2} on whole blocks once H~ Y_{k-1} is complete

Every arithmetic step runs in libchfsi kernels (binding.Operator); this module is bookkeeping plus the two collectives,
which go through a small communicator object so that the same code runs over NCCL (`TorchComm`) and, in the tests, in
one process that plays the ranks one after the other.  The exchange of one chunk can overlap the cell kernel of another:
`chebyshev_filter_chunked` keeps two chunks in flight ("asynchronous" boundary communication overlapped
with the compute of the next block)."""
from __future__ import annotations

from dataclasses import dataclass
from typing import List, Optional

import numpy as np


# ------------------------------------------------------------------------------------------------------------
# host-side partition (NumPy only; no device, no arithmetic of the method)
# ------------------------------------------------------------------------------------------------------------
@dataclass
class LocalPart:
    """What rank `rank` needs to create its operator: its cells with LOCAL dof ids, and its share of the projectors."""
    rank: int
    cells: np.ndarray              # [n_local_cells] global cell ids, ascending
    dofs: np.ndarray               # [n_local_dofs] global dof ids, ascending: local dof l <-> global dof dofs[l]
    cell_dofs: np.ndarray          # [n_local_cells, M_cell] int32, local ids
    cell_vertices: np.ndarray      # [n_local_cells, 8, 3]
    veff_q: np.ndarray             # [n_local_cells, n_q]
    proj_ids: np.ndarray           # [n_local_proj] global projector ids with at least one cell here, ascending
    D: np.ndarray                  # [n_local_proj]
    proj_cell_ptr: np.ndarray      # [n_local_proj + 1]
    proj_cell_idx: np.ndarray      # [nnz_local] LOCAL cell ids
    chi_q: np.ndarray              # [nnz_local, n_q]
    shared_rows: np.ndarray        # [n_shared_here] local rows of the dofs shared with other ranks, ascending
    shared_slots: np.ndarray       # [n_shared_here] their positions in the global list of shared dofs
    shared_owner: np.ndarray       # [n_shared_here] uint8: 1 where this rank is the lowest rank that holds the dof (its owner)


class CellPartition:
    """Cells split into `world` slabs of (nearly) equal size along the direction of largest extent, by centroid.
    Deterministic: every rank computes the same partition from the same mesh."""

    def __init__(self, wl, world: int):
        if world < 1:
            raise ValueError("world < 1")
        self.wl, self.world = wl, int(world)
        cd = np.asarray(wl.cell_dofs)
        nc = cd.shape[0]
        if world > nc:
            raise ValueError("more ranks than cells")
        cen = np.asarray(wl.cell_vertices).reshape(nc, 8, 3).mean(axis=1)
        axis = int(np.argmax(cen.max(axis=0) - cen.min(axis=0) + np.array([0.0, 1e-9, 2e-9])))   # ties: z, then y
        order = np.lexsort((np.arange(nc), np.round(cen[:, axis], 9)))
        self.owner = np.empty(nc, dtype=np.int32)
        for r in range(world):
            self.owner[order[(r * nc) // world:((r + 1) * nc) // world]] = r
        # ranks touching each dof
        touch = np.zeros((wl.n_dofs, world), dtype=bool)
        for r in range(world):
            touch[np.unique(cd[self.owner == r]), r] = True
        self.shared_dofs = np.nonzero(touch.sum(axis=1) >= 2)[0].astype(np.int64)     # global ids, ascending
        self._touch = touch
        self.n_proj = int(wl.n_proj)

    def local(self, rank: int) -> LocalPart:
        wl, cd = self.wl, np.asarray(self.wl.cell_dofs)
        cells = np.nonzero(self.owner == rank)[0]
        dofs = np.unique(cd[cells]).astype(np.int64)
        loc_cd = np.searchsorted(dofs, cd[cells]).astype(np.int32)
        cell_loc = -np.ones(cd.shape[0], dtype=np.int64)
        cell_loc[cells] = np.arange(len(cells))
        n_q = np.asarray(wl.veff_q).shape[1]
        ids, Dl, ptr, idx, chi = [], [], [0], [], []
        for j in range(self.n_proj):
            k0, k1 = int(wl.proj_cell_ptr[j]), int(wl.proj_cell_ptr[j + 1])
            here = [k for k in range(k0, k1) if self.owner[int(wl.proj_cell_idx[k])] == rank]
            if not here:
                continue
            ids.append(j); Dl.append(float(wl.D[j]))
            idx += [int(cell_loc[int(wl.proj_cell_idx[k])]) for k in here]
            chi += [np.asarray(wl.chi_q[k]) for k in here]
            ptr.append(len(idx))
        shared_here = self.shared_dofs[self._touch[self.shared_dofs, rank]]
        return LocalPart(
            rank=rank, cells=cells, dofs=dofs, cell_dofs=loc_cd,
            cell_vertices=np.ascontiguousarray(np.asarray(wl.cell_vertices).reshape(-1, 8, 3)[cells]),
            veff_q=np.ascontiguousarray(np.asarray(wl.veff_q)[cells]),
            proj_ids=np.asarray(ids, dtype=np.int64), D=np.asarray(Dl, dtype=np.float64),
            proj_cell_ptr=np.asarray(ptr, dtype=np.int64), proj_cell_idx=np.asarray(idx, dtype=np.int32),
            chi_q=np.asarray(chi, dtype=np.float64).reshape(len(idx), n_q),
            shared_rows=np.searchsorted(dofs, shared_here).astype(np.int32),
            shared_slots=np.searchsorted(self.shared_dofs, shared_here).astype(np.int32),
            shared_owner=(np.argmax(self._touch[shared_here], axis=1) == rank).astype(np.uint8))


# ------------------------------------------------------------------------------------------------------------
# communicators
# ------------------------------------------------------------------------------------------------------------
class TorchComm:
    """Sum over the ranks of a torch.distributed process group (NCCL for device tensors, gloo for host tensors)."""

    def __init__(self, group=None):
        import torch.distributed as dist
        self._dist, self.group = dist, group
        self.rank, self.world = dist.get_rank(group), dist.get_world_size(group)

    def all_reduce(self, t, async_op: bool = False):
        """In-place sum of a tensor; with async_op a handle whose wait() orders the current stream behind the collective."""
        return self._dist.all_reduce(t, op=self._dist.ReduceOp.SUM, group=self.group, async_op=async_op)

    def all_reduce_host(self, a: np.ndarray) -> np.ndarray:
        import torch
        dev = "cuda" if self._dist.get_backend(self.group) == "nccl" else "cpu"
        t = torch.from_numpy(np.ascontiguousarray(a)).to(dev)
        self._dist.all_reduce(t, op=self._dist.ReduceOp.SUM, group=self.group)
        return t.cpu().numpy()


class SingleComm:
    """world = 1: nothing to sum."""
    rank, world = 0, 1

    def all_reduce(self, t, async_op: bool = False):
        return None

    def all_reduce_host(self, a):
        return a


def global_mass_at(part: LocalPart, partition: CellPartition, p: int, comm) -> np.ndarray:
    """Diagonal mass of the WHOLE mesh at the part's dofs: chfsi_mesh_mass of the part's cells is complete on interior
    dofs; the shared dofs are summed over the ranks (one small host all-reduce at setup)."""
    from .binding import mesh_mass
    m = mesh_mass(p, part.cell_dofs, part.cell_vertices, len(part.dofs))
    buf = np.zeros(len(partition.shared_dofs), dtype=np.float64)
    buf[part.shared_slots] = m[part.shared_rows]
    buf = comm.all_reduce_host(buf)
    m[part.shared_rows] = buf[part.shared_slots]
    return m


# ------------------------------------------------------------------------------------------------------------
# the operator of one rank
# ------------------------------------------------------------------------------------------------------------
class PartitionedOperator:
    """The part of H~ that lives on this rank's cells + the two exchanges that complete it.

    Blocks are [n_local_dofs, B] device tensors (local row l = global dof part.dofs[l]); rows of shared dofs must hold the
    same values on every rank that has them (scatter_block does that for a global block).  boundary_fp32: the shared rows
    travel as FP32; every rank then unpacks the SAME rounded sums, so the replicas stay identical."""

    def __init__(self, wl, comm=None, precision: int = 64, assembly: int = 0, boundary_fp32: bool = False,
                 partition: Optional[CellPartition] = None, rank: Optional[int] = None, mass: Optional[np.ndarray] = None):
        import torch
        from .binding import Operator
        self.comm = comm if comm is not None else SingleComm()
        self.rank = self.comm.rank if rank is None else int(rank)
        self.partition = partition if partition is not None else CellPartition(wl, self.comm.world)
        self.part = self.partition.local(self.rank)
        pt = self.part
        self.mass = mass if mass is not None else global_mass_at(pt, self.partition, wl.p, self.comm)
        self.op = Operator(wl.p, pt.cell_dofs, pt.cell_vertices, len(pt.dofs), pt.veff_q, len(pt.proj_ids), pt.D,
                           pt.proj_cell_ptr, pt.proj_cell_idx, pt.chi_q, precision=precision, assembly=assembly,
                           dof_mass=self.mass)
        self.n_local_dofs = len(pt.dofs)
        self.n_proj_global = self.partition.n_proj
        self.n_shared = len(self.partition.shared_dofs)
        self.dtype = self.op.dtype
        self.payload_dtype = torch.float32 if boundary_fp32 else self.dtype
        dev = "cuda"
        self._rows = torch.from_numpy(pt.shared_rows).to(dev)
        self._slots = torch.from_numpy(pt.shared_slots).to(dev)
        self._owner = torch.from_numpy(pt.shared_owner).to(dev)
        self._proj_rows = torch.arange(len(pt.proj_ids), dtype=torch.int32, device=dev)
        self._proj_slots = torch.from_numpy(pt.proj_ids.astype(np.int32)).to(dev)

    # -- blocks ---------------------------------------------------------------------------------------------
    def scatter_block(self, X_global):
        """Rows of this rank from a global [n_dofs, B] host array or tensor -> [n_local_dofs, B] device tensor."""
        import torch
        Xg = torch.as_tensor(X_global)
        return Xg[torch.from_numpy(self.part.dofs)].to("cuda", self.dtype).contiguous()

    # -- the three local phases of one H~ application (the collectives sit between them) ----------------------
    def coefficients_partial(self, X, workspace=None):
        """[n_proj_global, B]: this rank's D C_part^T X in the rows of its projectors, zero elsewhere."""
        import torch
        B = int(X.shape[1])
        Pg = torch.zeros((max(self.n_proj_global, 1), B), dtype=self.dtype, device="cuda")
        if len(self.part.proj_ids):
            P = self.op.projector_coefficients(X, workspace=workspace)
            self.op.pack_rows(P, self._proj_rows, Pg, slots=self._proj_slots)
        return Pg

    def apply_partial(self, X, Pg, Y, workspace=None):
        """Y = this rank's contribution to H~ X (Pg summed over the ranks); returns the payload buffer [n_shared, B] with
        this rank's partial rows of the shared dofs in their slots, zero elsewhere."""
        import torch
        B = int(X.shape[1])
        P = torch.empty((len(self.part.proj_ids), B), dtype=self.dtype, device="cuda")
        if len(self.part.proj_ids):
            self.op.unpack_rows(Pg, self._proj_rows, P, slots=self._proj_slots)
        self.op.apply_H_with_coefficients(X, P, Y, workspace=workspace)
        buf = torch.zeros((max(self.n_shared, 1), B), dtype=self.payload_dtype, device="cuda")
        if self._rows.numel():
            self.op.pack_rows(Y, self._rows, buf, slots=self._slots)
        return buf

    def finish(self, Y, buf):
        """Rows of the shared dofs <- their sums over the ranks."""
        if self._rows.numel():
            self.op.unpack_rows(buf, self._rows, Y, slots=self._slots)
        return Y

    # -- whole operations -----------------------------------------------------------------------------------
    def apply_H(self, X, Y=None, workspace=None):
        import torch
        if Y is None:
            Y = torch.empty_like(X)
        Pg = self.coefficients_partial(X, workspace)
        self.comm.all_reduce(Pg)
        buf = self.apply_partial(X, Pg, Y, workspace)
        self.comm.all_reduce(buf)
        return self.finish(Y, buf)

    @staticmethod
    def recurrence_scalars(m, a, b, a0):
        """(alpha_k, beta_k) of the scaled three-term recurrence (U1) for k = 1 .. m, and the shift c."""
        e, c = 0.5 * (b - a), 0.5 * (b + a)
        s1 = e / (a0 - c)
        out, sg = [(s1 / e, 0.0)], s1
        for _ in range(2, m + 1):
            sn = 1.0 / (2.0 / s1 - sg)
            out.append((2.0 * sn / e, sg * sn))
            sg = sn
        return out, c

    def chebyshev_filter(self, X, m, a, b, a0, workspace=None):
        """In place on the local rows of a block (all ranks call it together)."""
        return self.chebyshev_filter_chunked(X, int(X.shape[1]), m, a, b, a0, workspace)

    @staticmethod
    def scaled_scalars(m, a, b, a0, precision=64):
        """The recurrence in scaled blocks W_k = s_k Y_k (U14; csrc/api.cu filter_block): W_1 = g_1 (H~ - c) W_0 and
        W_k = W_{k-2} + g_k (H~ - c) W_{k-1}; returns ([g_1 .. g_m], 1 / s_m, c), or None when |s_k| leaves the range of the
        storage type (the three-term form is used then)."""
        e, c = 0.5 * (b - a), 0.5 * (b + a)
        s1 = e / (a0 - c)
        limit = 1e200 if precision == 64 else 1e25
        gam, sg, s_km2, s_km1 = [s1 / e], s1, 1.0, 1.0
        for _ in range(2, m + 1):
            sn = 1.0 / (2.0 / s1 - sg)
            alpha, beta = 2.0 * sn / e, sg * sn
            sg = sn
            s_k = -s_km2 / beta
            if not (1.0 / limit < abs(s_k) < limit):
                return None
            gam.append(s_k * alpha / s_km1)
            s_km2, s_km1 = s_km1, s_k
        return gam, 1.0 / s_km1, c

    def chebyshev_filter_chunked(self, X, B, m, a, b, a0, workspace=None, scaled=True):
        """All N columns in chunks of B, TWO chunks in flight: while the shared rows of one chunk are on the wire (async
        all-reduce), the cell kernel of the other chunk runs.  scaled (default, where the part's kernel can add into its
        target block): the recurrence runs in scaled blocks, the cell kernel accumulates this part's contribution straight
        into W_{k-2} and only the shared rows are fixed up (pack_rows_delta / unpack_rows_sum) -- no recurrence pass over
        the block; otherwise H~X, the exchange and chfsi_recurrence_update."""
        import torch
        if m < 1 or not (a0 <= a < b):
            raise ValueError("need m >= 1 and a0 <= a < b")
        N = int(X.shape[1])
        B = min(int(B), N)
        scal, c = self.recurrence_scalars(m, a, b, a0)
        sc = self.scaled_scalars(m, a, b, a0, self.op.precision) if (scaled and m >= 2) else None
        ws = workspace if workspace is not None else self.op.workspace(B)
        chunks = [(j0, min(N, j0 + B)) for j0 in range(0, N, B)]
        n_here = int(self._rows.numel())
        for i0 in range(0, len(chunks), 2):
            pair = chunks[i0:i0 + 2]
            cur = [X[:, j0:j1] for j0, j1 in pair]                      # Y_{k-1}
            tgt = [torch.empty((self.n_local_dofs, j1 - j0), dtype=self.dtype, device="cuda") for j0, j1 in pair]   # Y_{k-2} -> Y_k
            if sc is not None and all(self.op.accumulate_supported(cur[q], tgt[q], ws) for q in range(len(pair))):
                gam, inv_sm, _ = sc
                for k, g in enumerate(gam, start=1):
                    bufs, works, bases = [], [], []
                    for q in range(len(pair)):
                        Bq = int(cur[q].shape[1])
                        Pg = self.coefficients_partial(cur[q], ws)
                        self.comm.all_reduce(Pg)
                        P = torch.empty((len(self.part.proj_ids), Bq), dtype=self.dtype, device="cuda")
                        if len(self.part.proj_ids):
                            self.op.unpack_rows(Pg, self._proj_rows, P, slots=self._proj_slots)
                        base = None
                        if k >= 2 and n_here:                             # the shared rows of W_{k-2} before this part adds to them
                            base = torch.empty((n_here, Bq), dtype=self.dtype, device="cuda")
                            self.op.pack_rows(tgt[q], self._rows, base)
                        self.op.apply_shifted_with_coefficients(cur[q], P, tgt[q], g, c, k >= 2, workspace=ws)
                        buf = torch.zeros((max(self.n_shared, 1), Bq), dtype=self.payload_dtype, device="cuda")
                        if n_here:
                            self.op.pack_rows_delta(tgt[q], base, cur[q], self._owner, g * c, self._rows, buf, slots=self._slots)
                        works.append(self.comm.all_reduce(buf, async_op=True))
                        bufs.append(buf); bases.append(base)
                    for q in range(len(pair)):
                        if works[q] is not None:
                            works[q].wait()
                        if n_here:
                            self.op.unpack_rows_sum(bufs[q], bases[q], self._rows, tgt[q], slots=self._slots)
                        cur[q], tgt[q] = tgt[q], cur[q]
                for q, (j0, j1) in enumerate(pair):                      # X <- W_m / s_m (in place when m is even)
                    out = X[:, j0:j1]
                    self.op.recurrence_update(cur[q], cur[q], out, inv_sm, 0.0, 0.0)
                continue
            HX = [torch.empty_like(t) for t in tgt]
            for alpha, beta in scal:
                bufs, works = [], []
                for q in range(len(pair)):
                    Pg = self.coefficients_partial(cur[q], ws)
                    self.comm.all_reduce(Pg)
                    buf = self.apply_partial(cur[q], Pg, HX[q], ws)
                    works.append(self.comm.all_reduce(buf, async_op=True))   # chunk q on the wire while chunk q + 1 computes
                    bufs.append(buf)
                for q in range(len(pair)):
                    if works[q] is not None:
                        works[q].wait()
                    self.finish(HX[q], bufs[q])
                    self.op.recurrence_update(HX[q], cur[q], tgt[q], alpha, beta, c)
                    cur[q], tgt[q] = tgt[q], cur[q]
            for q, (j0, j1) in enumerate(pair):
                if cur[q].data_ptr() != X[:, j0:j1].data_ptr():
                    X[:, j0:j1].copy_(cur[q])
        return X

    def close(self):
        self.op.close()
