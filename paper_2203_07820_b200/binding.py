"""ctypes binding of libchfsi (include/chfsi.h).  Argument marshalling only.

`Operator` mirrors the C entry points one to one:
    chfsi_create / chfsi_destroy / chfsi_get_info / chfsi_workspace_bytes / chfsi_mass_diag /
    chfsi_apply_H / chfsi_chebyshev_filter / chfsi_chebyshev_filter_chunked / chfsi_chebyshev_filter_host /
    chfsi_launch_count / chfsi_set_kernel_variant / chfsi_last_error
Vector blocks are torch CUDA tensors of shape [n_dofs, ld] (row-major, vector index fastest);
a chunk of columns is passed as a column slice `X[:, j0:j0+B]` (stride(0) = ld, stride(1) = 1).
"""
from __future__ import annotations

import ctypes as C
import os
from typing import Optional

import numpy as np

HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(HERE, "libchfsi.so")

EXPORTED_SYMBOLS = [
    "chfsi_create", "chfsi_create_k", "chfsi_create_part", "chfsi_mesh_mass", "chfsi_projector_coefficients",
    "chfsi_apply_H_with_coefficients", "chfsi_pack_rows", "chfsi_unpack_rows", "chfsi_recurrence_update", "chfsi_accumulate_supported", "chfsi_apply_shifted_with_coefficients",
    "chfsi_pack_rows_delta", "chfsi_unpack_rows_sum", "chfsi_destroy", "chfsi_update_potential", "chfsi_get_info", "chfsi_workspace_bytes", "chfsi_mass_diag",
    "chfsi_apply_H", "chfsi_overlap_matrix", "chfsi_overlap_matrix_noalloc", "chfsi_projected_hamiltonian", "chfsi_subspace_transform",
    "chfsi_cholesky_inverse", "chfsi_overlap_matrix_mixed", "chfsi_projected_hamiltonian_mixed", "chfsi_subspace_transform_mixed", "chfsi_chebyshev_filter", "chfsi_chebyshev_filter_chunked", "chfsi_chebyshev_filter_host",
    "chfsi_launch_count", "chfsi_set_kernel_variant", "chfsi_set_rr_variant", "chfsi_set_profiling", "chfsi_get_profile",
    "chfsi_measure_fp64_peak", "chfsi_last_error",
]


class ChfsiError(RuntimeError):
    def __init__(self, code: int, msg: str):
        super().__init__(f"libchfsi error {code}: {msg}")
        self.code = code


class _KPoint(C.Structure):
    _fields_ = [("k", C.c_double * 3), ("chi_q_im", C.c_void_p)]


class _Mesh(C.Structure):
    _fields_ = [("p", C.c_int32), ("n_cells", C.c_int64), ("n_dofs", C.c_int64),
                ("cell_dofs", C.c_void_p), ("cell_vertices", C.c_void_p)]


class _Potential(C.Structure):
    _fields_ = [("veff_q", C.c_void_p)]


class _Nonlocal(C.Structure):
    _fields_ = [("n_proj", C.c_int64), ("D", C.c_void_p), ("proj_cell_ptr", C.c_void_p),
                ("proj_cell_idx", C.c_void_p), ("chi_q", C.c_void_p)]


class _Info(C.Structure):
    _fields_ = [("p", C.c_int32), ("m_cell", C.c_int32), ("n_q", C.c_int32), ("precision", C.c_int32),
                ("assembly", C.c_int32), ("n_colors", C.c_int32),
                ("n_cells", C.c_int64), ("n_dofs", C.c_int64), ("n_proj", C.c_int64),
                ("nnz_cell_proj", C.c_int64), ("cells_with_proj", C.c_int64),
                ("flops_per_vector_apply", C.c_double), ("matrix_bytes", C.c_int64),
                ("sf_flops_per_vector_apply", C.c_double), ("sf_field_bytes", C.c_int64)]


class _Profile(C.Structure):
    _fields_ = [("contraction_ms", C.c_double), ("contraction_launches", C.c_int64),
                ("projector_ms", C.c_double), ("projector_launches", C.c_int64), ("applies", C.c_int64)]


_lib = None


def load_library(build_if_missing: bool = True):
    """dlopen libchfsi.so (building it in-tree with nvcc first if it is missing or stale)."""
    global _lib
    if _lib is not None:
        return _lib
    if build_if_missing:
        from .build import build
        build()
    if not os.path.exists(LIB_PATH):
        raise RuntimeError(f"{LIB_PATH} is missing: build it with `python -m paper_2203_07820_b200.build` "
                           "(there is no CPU fallback)")
    lib_ = C.CDLL(LIB_PATH)
    vp, i64, i32, dbl = C.c_void_p, C.c_int64, C.c_int32, C.c_double
    lib_.chfsi_create.argtypes = [C.POINTER(vp), C.POINTER(_Mesh), C.POINTER(_Potential), C.POINTER(_Nonlocal),
                                  C.c_int, C.c_int, vp]
    lib_.chfsi_create.restype = C.c_int
    lib_.chfsi_create_k.argtypes = [C.POINTER(vp), C.POINTER(_Mesh), C.POINTER(_Potential), C.POINTER(_Nonlocal),
                                    C.POINTER(_KPoint), C.c_int, vp]
    lib_.chfsi_create_k.restype = C.c_int
    lib_.chfsi_create_part.argtypes = [C.POINTER(vp), C.POINTER(_Mesh), C.POINTER(_Potential), C.POINTER(_Nonlocal), vp,
                                       C.c_int, C.c_int, vp]
    lib_.chfsi_create_part.restype = C.c_int
    lib_.chfsi_mesh_mass.argtypes = [C.POINTER(_Mesh), vp]
    lib_.chfsi_mesh_mass.restype = C.c_int
    lib_.chfsi_projector_coefficients.argtypes = [vp, vp, i64, i64, vp, vp, vp]
    lib_.chfsi_projector_coefficients.restype = C.c_int
    lib_.chfsi_apply_H_with_coefficients.argtypes = [vp, vp, i64, vp, i64, i64, vp, vp, vp]
    lib_.chfsi_apply_H_with_coefficients.restype = C.c_int
    lib_.chfsi_pack_rows.argtypes = [vp, vp, i64, i64, vp, vp, i64, vp, C.c_int, vp]
    lib_.chfsi_pack_rows.restype = C.c_int
    lib_.chfsi_unpack_rows.argtypes = [vp, vp, C.c_int, vp, vp, i64, vp, i64, i64, vp]
    lib_.chfsi_unpack_rows.restype = C.c_int
    lib_.chfsi_recurrence_update.argtypes = [vp, vp, i64, vp, i64, vp, i64, i64, dbl, dbl, dbl, vp]
    lib_.chfsi_recurrence_update.restype = C.c_int
    lib_.chfsi_accumulate_supported.argtypes = [vp, vp, i64, vp, i64, i64, vp, C.POINTER(C.c_int)]
    lib_.chfsi_accumulate_supported.restype = C.c_int
    lib_.chfsi_apply_shifted_with_coefficients.argtypes = [vp, vp, i64, vp, i64, i64, dbl, dbl, C.c_int, vp, vp, vp]
    lib_.chfsi_apply_shifted_with_coefficients.restype = C.c_int
    lib_.chfsi_pack_rows_delta.argtypes = [vp, vp, i64, vp, vp, i64, vp, dbl, i64, vp, vp, i64, vp, C.c_int, vp]
    lib_.chfsi_pack_rows_delta.restype = C.c_int
    lib_.chfsi_unpack_rows_sum.argtypes = [vp, vp, C.c_int, vp, vp, vp, i64, vp, i64, i64, vp]
    lib_.chfsi_unpack_rows_sum.restype = C.c_int
    lib_.chfsi_destroy.argtypes = [vp]
    lib_.chfsi_destroy.restype = C.c_int
    lib_.chfsi_update_potential.argtypes = [vp, C.POINTER(_Potential), vp]
    lib_.chfsi_update_potential.restype = C.c_int
    lib_.chfsi_get_info.argtypes = [vp, C.POINTER(_Info)]
    lib_.chfsi_get_info.restype = C.c_int
    lib_.chfsi_workspace_bytes.argtypes = [vp, i64, C.POINTER(C.c_size_t)]
    lib_.chfsi_workspace_bytes.restype = C.c_int
    lib_.chfsi_mass_diag.argtypes = [vp, vp, vp]
    lib_.chfsi_mass_diag.restype = C.c_int
    lib_.chfsi_apply_H.argtypes = [vp, vp, i64, vp, i64, i64, vp, vp]
    lib_.chfsi_apply_H.restype = C.c_int
    lib_.chfsi_overlap_matrix.argtypes = [vp, vp, i64, i64, vp, vp]
    lib_.chfsi_overlap_matrix.restype = C.c_int
    lib_.chfsi_overlap_matrix_noalloc.argtypes = [vp, vp, i64, i64, vp, vp]
    lib_.chfsi_overlap_matrix_noalloc.restype = C.c_int
    lib_.chfsi_projected_hamiltonian.argtypes = [vp, vp, i64, i64, i64, vp, vp, vp]
    lib_.chfsi_projected_hamiltonian.restype = C.c_int
    lib_.chfsi_subspace_transform.argtypes = [vp, vp, i64, i64, vp, i64, i64, vp, i64, vp]
    lib_.chfsi_subspace_transform.restype = C.c_int
    lib_.chfsi_cholesky_inverse.argtypes = [vp, vp, i64, vp, vp, vp, vp]
    lib_.chfsi_cholesky_inverse.restype = C.c_int
    lib_.chfsi_overlap_matrix_mixed.argtypes = [vp, vp, i64, i64, i64, vp, vp]
    lib_.chfsi_overlap_matrix_mixed.restype = C.c_int
    lib_.chfsi_projected_hamiltonian_mixed.argtypes = [vp, vp, i64, i64, i64, i64, vp, vp, vp]
    lib_.chfsi_projected_hamiltonian_mixed.restype = C.c_int
    lib_.chfsi_subspace_transform_mixed.argtypes = [vp, vp, i64, i64, vp, i64, vp, i64, vp]
    lib_.chfsi_subspace_transform_mixed.restype = C.c_int
    lib_.chfsi_chebyshev_filter.argtypes = [vp, vp, i64, i64, i32, dbl, dbl, dbl, vp, vp]
    lib_.chfsi_chebyshev_filter.restype = C.c_int
    lib_.chfsi_chebyshev_filter_chunked.argtypes = [vp, vp, i64, i64, i64, i32, dbl, dbl, dbl, vp, vp]
    lib_.chfsi_chebyshev_filter_chunked.restype = C.c_int
    lib_.chfsi_chebyshev_filter_host.argtypes = [vp, vp, i64, i64, i64, i32, dbl, dbl, dbl]
    lib_.chfsi_chebyshev_filter_host.restype = C.c_int
    lib_.chfsi_launch_count.argtypes = [vp]
    lib_.chfsi_launch_count.restype = i64
    lib_.chfsi_set_kernel_variant.argtypes = [vp, C.c_int]
    lib_.chfsi_set_kernel_variant.restype = C.c_int
    lib_.chfsi_set_rr_variant.argtypes = [vp, C.c_int]
    lib_.chfsi_set_rr_variant.restype = C.c_int
    lib_.chfsi_set_profiling.argtypes = [vp, C.c_int]
    lib_.chfsi_set_profiling.restype = C.c_int
    lib_.chfsi_get_profile.argtypes = [vp, C.POINTER(_Profile)]
    lib_.chfsi_get_profile.restype = C.c_int
    lib_.chfsi_measure_fp64_peak.argtypes = [C.POINTER(dbl), C.POINTER(dbl), vp]
    lib_.chfsi_measure_fp64_peak.restype = C.c_int
    lib_.chfsi_last_error.argtypes = [vp]
    lib_.chfsi_last_error.restype = C.c_char_p
    _lib = lib_
    return _lib


def lib():
    return load_library()


def _np_ptr(a: np.ndarray) -> int:
    return a.ctypes.data


def _stream_ptr(stream) -> Optional[int]:
    import torch
    s = stream if stream is not None else torch.cuda.current_stream()
    return C.c_void_p(s.cuda_stream)


def measure_fp64_peak(stream=None) -> dict:
    """{'dmma_tflops', 'dfma_tflops'} of the current device (chfsi_measure_fp64_peak)."""
    a, b = C.c_double(), C.c_double()
    rc = load_library().chfsi_measure_fp64_peak(C.byref(a), C.byref(b), _stream_ptr(stream))
    if rc != 0:
        raise ChfsiError(rc, "chfsi_measure_fp64_peak failed")
    return {"dmma_tflops": a.value, "dfma_tflops": b.value}


def mesh_mass(p, cell_dofs, cell_vertices, n_dofs) -> np.ndarray:
    """chfsi_mesh_mass: diagonal GLL mass of a mesh (or of a part of one: the partial sums over its cells).  Host only."""
    cell_dofs = np.ascontiguousarray(cell_dofs, dtype=np.int32)
    cell_vertices = np.ascontiguousarray(cell_vertices, dtype=np.float64)
    mesh = _Mesh(int(p), int(cell_dofs.shape[0]), int(n_dofs), _np_ptr(cell_dofs), _np_ptr(cell_vertices))
    M = np.empty(int(n_dofs), dtype=np.float64)
    rc = load_library().chfsi_mesh_mass(C.byref(mesh), M.ctypes.data)
    if rc != 0:
        raise ChfsiError(rc, (load_library().chfsi_last_error(None) or b"").decode())
    return M


class Operator:
    """Owns one `chfsi_op` handle.  Inputs are host NumPy arrays (copied by the library during the call)."""

    def __init__(self, p, cell_dofs, cell_vertices, n_dofs, veff_q, n_proj=0, D=None, proj_cell_ptr=None,
                 proj_cell_idx=None, chi_q=None, precision=64, assembly=0, stream=None, kvec=None, chi_q_im=None,
                 dof_mass=None):
        """kvec (3 floats, bohr^-1) selects the k-point variant (chfsi_create_k): blocks are then complex128 tensors and
        chi_q / chi_q_im hold the real / imaginary parts of the Bloch-phased projector samples.  dof_mass ([n_dofs], the
        diagonal mass of the whole mesh at these dofs) makes the handle a PART of a larger mesh (chfsi_create_part)."""
        self._h = None
        self.kpoint = kvec is not None
        L = load_library()
        import torch
        if not torch.cuda.is_available():
            raise ChfsiError(-4, "no CUDA device: libchfsi has no CPU fallback")
        cell_dofs = np.ascontiguousarray(cell_dofs, dtype=np.int32)
        cell_vertices = np.ascontiguousarray(cell_vertices, dtype=np.float64)
        veff_q = np.ascontiguousarray(veff_q, dtype=np.float64)
        mesh = _Mesh(int(p), int(cell_dofs.shape[0]), int(n_dofs), _np_ptr(cell_dofs), _np_ptr(cell_vertices))
        pot = _Potential(_np_ptr(veff_q))
        keep = [cell_dofs, cell_vertices, veff_q]
        nlp = None
        if n_proj:
            D = np.ascontiguousarray(D, dtype=np.float64)
            ptr = np.ascontiguousarray(proj_cell_ptr, dtype=np.int64)
            idx = np.ascontiguousarray(proj_cell_idx, dtype=np.int32)
            chi = np.ascontiguousarray(chi_q, dtype=np.float64)
            keep += [D, ptr, idx, chi]
            nlp = C.pointer(_Nonlocal(int(n_proj), _np_ptr(D), _np_ptr(ptr), _np_ptr(idx), _np_ptr(chi)))
        h = C.c_void_p()
        if self.kpoint:
            kp = _KPoint()
            for i in range(3):
                kp.k[i] = float(kvec[i])
            if n_proj:
                chi_im = np.ascontiguousarray(chi_q_im if chi_q_im is not None else np.zeros_like(chi), dtype=np.float64)
                keep.append(chi_im)
                kp.chi_q_im = chi_im.ctypes.data
            rc = L.chfsi_create_k(C.byref(h), C.byref(mesh), C.byref(pot), nlp, C.byref(kp), int(assembly),
                                  _stream_ptr(stream))
        elif dof_mass is not None:
            dm = np.ascontiguousarray(dof_mass, dtype=np.float64)
            if dm.shape != (int(n_dofs),):
                raise ValueError("dof_mass must have n_dofs entries")
            rc = L.chfsi_create_part(C.byref(h), C.byref(mesh), C.byref(pot), nlp, dm.ctypes.data, int(precision),
                                     int(assembly), _stream_ptr(stream))
        else:
            rc = L.chfsi_create(C.byref(h), C.byref(mesh), C.byref(pot), nlp, int(precision), int(assembly),
                                _stream_ptr(stream))
        if rc != 0:
            raise ChfsiError(rc, (L.chfsi_last_error(None) or b"").decode())
        self._h = h
        self.precision = int(precision)
        info = _Info()
        self._check(L.chfsi_get_info(self._h, C.byref(info)))
        self.info = {k: getattr(info, k) for k, _ in _Info._fields_}
        self.n_dofs = int(info.n_dofs)
        self._ws = None
        self._ws_B = 0

    @classmethod
    def from_workload(cls, wl, precision=64, assembly=0, stream=None):
        """wl.kvec set (workloads.generate.make_workload(kvec=...)): the k-point variant."""
        return cls(wl.p, wl.cell_dofs, wl.cell_vertices, wl.n_dofs, wl.veff_q, wl.n_proj, wl.D, wl.proj_cell_ptr,
                   wl.proj_cell_idx, wl.chi_q, precision=precision, assembly=assembly, stream=stream,
                   kvec=getattr(wl, "kvec", None), chi_q_im=getattr(wl, "chi_q_im", None))

    # -- helpers ------------------------------------------------------------------------------------------
    def _check(self, rc: int):
        if rc != 0:
            raise ChfsiError(rc, (load_library().chfsi_last_error(self._h) or b"").decode())

    @property
    def dtype(self):
        import torch
        if self.kpoint:
            return torch.complex128
        return torch.float64 if self.precision == 64 else torch.float32

    def _block(self, X, name):
        import torch
        if not (isinstance(X, torch.Tensor) and X.is_cuda and X.dim() == 2):
            raise TypeError(f"{name}: expected a 2-D CUDA tensor [n_dofs, B]")
        if X.dtype != self.dtype:
            raise TypeError(f"{name}: dtype {X.dtype} does not match operator precision {self.precision}")
        if X.shape[0] != self.n_dofs or X.stride(1) != 1 or X.stride(0) < X.shape[1]:
            raise ValueError(f"{name}: need shape [n_dofs, B] with the vector index fastest")
        return C.c_void_p(X.data_ptr()), int(X.stride(0)), int(X.shape[1])

    def workspace_bytes(self, B: int) -> int:
        n = C.c_size_t()
        self._check(load_library().chfsi_workspace_bytes(self._h, int(B), C.byref(n)))
        return int(n.value)

    def workspace(self, B: int):
        """A cached torch-allocated device workspace for blocks of B columns."""
        import torch
        if self._ws is None or self._ws_B != B:
            self._ws = None
            self._ws = torch.empty(self.workspace_bytes(B), dtype=torch.uint8, device="cuda")
            self._ws_B = B
        return self._ws

    # -- the ABI calls ------------------------------------------------------------------------------------
    def mass_diag(self, stream=None):
        import torch
        M = torch.empty(self.n_dofs, dtype=torch.float64, device="cuda")
        self._check(load_library().chfsi_mass_diag(self._h, C.c_void_p(M.data_ptr()), _stream_ptr(stream)))
        return M

    def apply_H(self, X, Y=None, workspace=None, stream=None):
        import torch
        xp, ldx, B = self._block(X, "X")
        if Y is None:
            Y = torch.empty((self.n_dofs, B), dtype=self.dtype, device="cuda")
        yp, ldy, By = self._block(Y, "Y")
        if By != B:
            raise ValueError("X and Y must have the same number of columns")
        ws = workspace if workspace is not None else self.workspace(B)
        self._check(load_library().chfsi_apply_H(self._h, xp, ldx, yp, ldy, B, C.c_void_p(ws.data_ptr()),
                                                 _stream_ptr(stream)))
        return Y

    # -- cell-partitioned operation (include/chfsi.h "Cell-partitioned operation") --------------------------------
    def projector_coefficients(self, X, P=None, workspace=None, stream=None):
        """P[n_proj, B] = D (C^T X) over this operator's cells (steps 3a-3c); a device tensor of the operator's dtype."""
        import torch
        xp, ldx, B = self._block(X, "X")
        n_proj = int(self.info["n_proj"])
        if P is None:
            P = torch.zeros((n_proj, B), dtype=self.dtype, device="cuda")
        if tuple(P.shape) != (n_proj, B) or not P.is_contiguous() or P.dtype != self.dtype:
            raise ValueError("P must be a contiguous [n_proj, B] tensor of the operator's dtype")
        ws = workspace if workspace is not None else self.workspace(B)
        self._check(load_library().chfsi_projector_coefficients(self._h, xp, ldx, B, C.c_void_p(P.data_ptr()),
                                                                C.c_void_p(ws.data_ptr()), _stream_ptr(stream)))
        return P

    def apply_H_with_coefficients(self, X, P, Y=None, workspace=None, stream=None):
        """This operator's contribution to H~ X with the projector coefficients P[n_proj, B] given."""
        import torch
        xp, ldx, B = self._block(X, "X")
        if Y is None:
            Y = torch.empty((self.n_dofs, B), dtype=self.dtype, device="cuda")
        yp, ldy, By = self._block(Y, "Y")
        n_proj = int(self.info["n_proj"])
        if By != B or tuple(P.shape) != (n_proj, B) or not P.is_contiguous() or P.dtype != self.dtype:
            raise ValueError("need Y [n_dofs, B] and a contiguous P [n_proj, B] of the operator's dtype")
        ws = workspace if workspace is not None else self.workspace(B)
        self._check(load_library().chfsi_apply_H_with_coefficients(self._h, xp, ldx, yp, ldy, B, C.c_void_p(P.data_ptr()),
                                                                   C.c_void_p(ws.data_ptr()), _stream_ptr(stream)))
        return Y

    def _rows_block(self, X, name):
        import torch
        if not (isinstance(X, torch.Tensor) and X.is_cuda and X.dim() == 2 and X.dtype == self.dtype and X.stride(1) == 1):
            raise TypeError(f"{name}: expected a 2-D CUDA tensor of the operator's dtype, vector index fastest")
        return C.c_void_p(X.data_ptr()), int(X.stride(0)), int(X.shape[1])

    def pack_rows(self, X, rows, buf, slots=None, stream=None):
        """buf[s(i)] = X[rows[i]], s(i) = slots[i] or i (rows, slots: int32 device tensors; buf: contiguous [., B] of X's dtype
        or float32)."""
        import torch
        xp, ldx, B = self._rows_block(X, "X")
        bp = 32 if buf.dtype == torch.float32 else 64
        sp = C.c_void_p(slots.data_ptr()) if slots is not None else None
        self._check(load_library().chfsi_pack_rows(self._h, xp, ldx, B, C.c_void_p(rows.data_ptr()), sp, int(rows.numel()),
                                                   C.c_void_p(buf.data_ptr()), bp, _stream_ptr(stream)))
        return buf

    def unpack_rows(self, buf, rows, X, slots=None, stream=None):
        """X[rows[i]] = buf[s(i)]."""
        import torch
        xp, ldx, B = self._rows_block(X, "X")
        bp = 32 if buf.dtype == torch.float32 else 64
        sp = C.c_void_p(slots.data_ptr()) if slots is not None else None
        self._check(load_library().chfsi_unpack_rows(self._h, C.c_void_p(buf.data_ptr()), bp, C.c_void_p(rows.data_ptr()), sp,
                                                     int(rows.numel()), xp, ldx, B, _stream_ptr(stream)))
        return X

    def recurrence_update(self, HX, X, T, alpha, beta, c, stream=None):
        """T <- alpha (HX - c X) - beta T on whole blocks."""
        hp, ldh, B = self._block(HX, "HX")
        xp, ldx, Bx = self._block(X, "X")
        tp, ldt, Bt = self._block(T, "T")
        if not (B == Bx == Bt):
            raise ValueError("HX, X and T must have the same number of columns")
        self._check(load_library().chfsi_recurrence_update(self._h, hp, ldh, xp, ldx, tp, ldt, B, float(alpha), float(beta),
                                                           float(c), _stream_ptr(stream)))
        return T

    # -- the exchange of the filter in scaled (accumulate-only) blocks: include/chfsi.h ----------------------------
    def accumulate_supported(self, X, T, workspace=None) -> bool:
        """True when apply_shifted_with_coefficients(..., accumulate=True) is available for these blocks."""
        xp, ldx, B = self._block(X, "X")
        tp, ldt, Bt = self._block(T, "T")
        if B != Bt:
            raise ValueError("X and T must have the same number of columns")
        ws = workspace if workspace is not None else self.workspace(B)
        yes = C.c_int(0)
        self._check(load_library().chfsi_accumulate_supported(self._h, xp, ldx, tp, ldt, B, C.c_void_p(ws.data_ptr()), C.byref(yes)))
        return bool(yes.value)

    def apply_shifted_with_coefficients(self, X, P, T, alpha, c, accumulate, workspace=None, stream=None):
        """T = alpha (H~_part - c) X (accumulate False) or T += alpha (H~_part - c) X, projector coefficients P given."""
        xp, ldx, B = self._block(X, "X")
        tp, ldt, Bt = self._block(T, "T")
        n_proj = int(self.info["n_proj"])
        if Bt != B or tuple(P.shape) != (n_proj, B) or not P.is_contiguous() or P.dtype != self.dtype:
            raise ValueError("need T [n_dofs, B] and a contiguous P [n_proj, B] of the operator's dtype")
        ws = workspace if workspace is not None else self.workspace(B)
        self._check(load_library().chfsi_apply_shifted_with_coefficients(
            self._h, xp, ldx, tp, ldt, B, float(alpha), float(c), 1 if accumulate else 0, C.c_void_p(P.data_ptr()),
            C.c_void_p(ws.data_ptr()), _stream_ptr(stream)))
        return T

    def pack_rows_delta(self, T, base, X, owner, corr, rows, buf, slots=None, stream=None):
        """buf[s(i)] = T[rows[i]] - base[i] + corr X[rows[i]] (1 - owner[i]); base: contiguous [n_rows, B] or None; owner: uint8."""
        import torch
        tp, ldt, B = self._rows_block(T, "T")
        xp, ldx, Bx = self._rows_block(X, "X")
        n = int(rows.numel())
        if Bx != B or owner.dtype != torch.uint8 or int(owner.numel()) != n:
            raise ValueError("need X with T's columns and one uint8 owner flag per row")
        if base is not None and not (base.is_contiguous() and tuple(base.shape) == (n, B) and base.dtype == T.dtype):
            raise ValueError("base: contiguous [n_rows, B] of T's dtype")
        bp = 32 if buf.dtype == torch.float32 else 64
        sp = C.c_void_p(slots.data_ptr()) if slots is not None else None
        bs = C.c_void_p(base.data_ptr()) if base is not None else None
        self._check(load_library().chfsi_pack_rows_delta(self._h, tp, ldt, bs, xp, ldx, C.c_void_p(owner.data_ptr()), float(corr), B,
                                                         C.c_void_p(rows.data_ptr()), sp, n, C.c_void_p(buf.data_ptr()), bp,
                                                         _stream_ptr(stream)))
        return buf

    def unpack_rows_sum(self, buf, base, rows, T, slots=None, stream=None):
        """T[rows[i]] = base[i] + buf[s(i)] (base None: 0)."""
        import torch
        tp, ldt, B = self._rows_block(T, "T")
        n = int(rows.numel())
        if base is not None and not (base.is_contiguous() and tuple(base.shape) == (n, B) and base.dtype == T.dtype):
            raise ValueError("base: contiguous [n_rows, B] of T's dtype")
        bp = 32 if buf.dtype == torch.float32 else 64
        sp = C.c_void_p(slots.data_ptr()) if slots is not None else None
        bs = C.c_void_p(base.data_ptr()) if base is not None else None
        self._check(load_library().chfsi_unpack_rows_sum(self._h, C.c_void_p(buf.data_ptr()), bp, bs, C.c_void_p(rows.data_ptr()), sp, n,
                                                         tp, ldt, B, _stream_ptr(stream)))
        return T

    def overlap_matrix(self, Y, stream=None):
        """S = Y^T Y (Algorithm 2 step 1a); returns a [N, N] FP64 device tensor."""
        import torch
        yp, ldy, N = self._block(Y, "Y")
        S = torch.empty((N, N), dtype=torch.float64, device="cuda")
        self._check(load_library().chfsi_overlap_matrix(self._h, yp, ldy, N, C.c_void_p(S.data_ptr()),
                                                        _stream_ptr(stream)))
        return S

    def overlap_matrix_noalloc(self, Y, S, stream=None):
        """S <- Y^T Y through chfsi_overlap_matrix_noalloc: the library allocates nothing (static scratch, N <= 512; calls
        that overlap on the GPU race on it).  `S` is the caller's contiguous [N, N] FP64 device tensor."""
        import torch
        yp, ldy, N = self._block(Y, "Y")
        if not (isinstance(S, torch.Tensor) and S.is_cuda and S.dtype == torch.float64 and S.shape == (N, N) and S.is_contiguous()):
            raise TypeError("S: expected a contiguous [N, N] float64 CUDA tensor")
        self._check(load_library().chfsi_overlap_matrix_noalloc(self._h, yp, ldy, N, C.c_void_p(S.data_ptr()),
                                                                _stream_ptr(stream)))
        return S

    def projected_hamiltonian(self, Y, B=None, workspace=None, stream=None):
        """H^ = Y^T (H~ Y) (Algorithm 2 step 1b), H~ Y formed B columns at a time; returns [N, N] FP64."""
        import torch
        yp, ldy, N = self._block(Y, "Y")
        B = int(B) if B is not None else min(N, 256)
        ws = workspace if workspace is not None else self.workspace(min(B, N))
        Hh = torch.empty((N, N), dtype=torch.float64, device="cuda")
        self._check(load_library().chfsi_projected_hamiltonian(self._h, yp, ldy, N, B, C.c_void_p(Hh.data_ptr()),
                                                               C.c_void_p(ws.data_ptr()), _stream_ptr(stream)))
        return Hh

    def subspace_transform(self, Y, Z, Out=None, stream=None):
        """Out = Y Z (Algorithm 2 step 3); Z is a [N, N2] FP64 device tensor (row-major)."""
        import torch
        yp, ldy, N = self._block(Y, "Y")
        if Z.dim() != 2 or Z.shape[0] != N or Z.dtype != torch.float64 or Z.stride(1) != 1 or not Z.is_cuda:
            raise ValueError("Z must be a [N, N2] FP64 CUDA tensor with unit column stride")
        N2 = int(Z.shape[1])
        if Out is None:
            Out = torch.empty((self.n_dofs, N2), dtype=torch.float64, device="cuda")
        op_, ldo, No = self._block(Out, "Out")
        if No != N2:
            raise ValueError("Out must have N2 columns")
        self._check(load_library().chfsi_subspace_transform(self._h, yp, ldy, N, C.c_void_p(Z.data_ptr()),
                                                            int(Z.stride(0)), N2, op_, ldo, _stream_ptr(stream)))
        return Out

    def cholesky_inverse(self, S, stream=None):
        """Algorithm 2 step 2a on the device: returns (L, L^-1, info) for S = L L^T; info is a device int32 tensor
        (0 = success, else the 1-based index of the first non-positive pivot)."""
        import torch
        if not (S.is_cuda and S.dim() == 2 and S.shape[0] == S.shape[1] and S.dtype == torch.float64 and S.is_contiguous()):
            raise ValueError("S must be a contiguous square FP64 CUDA tensor")
        N = int(S.shape[0])
        L, Linv = torch.empty_like(S), torch.empty_like(S)
        info = torch.zeros(1, dtype=torch.int32, device="cuda")
        self._check(load_library().chfsi_cholesky_inverse(self._h, C.c_void_p(S.data_ptr()), N, C.c_void_p(L.data_ptr()),
                                                          C.c_void_p(Linv.data_ptr()), C.c_void_p(info.data_ptr()),
                                                          _stream_ptr(stream)))
        return L, Linv, info

    def overlap_matrix_mixed(self, Y, block, stream=None):
        """S = Y^T Y, diagonal blocks of width `block` FP64, the rest FP32."""
        import torch
        yp, ldy, N = self._block(Y, "Y")
        S = torch.empty((N, N), dtype=torch.float64, device="cuda")
        self._check(load_library().chfsi_overlap_matrix_mixed(self._h, yp, ldy, N, int(block), C.c_void_p(S.data_ptr()),
                                                              _stream_ptr(stream)))
        return S

    def projected_hamiltonian_mixed(self, Y, n_oc, B=None, workspace=None, stream=None):
        """H^ = Y^T (H~ Y) with the blocking of Eq. 39: fr-fr block (rows, columns >= n_oc) FP64, the rest FP32."""
        import torch
        yp, ldy, N = self._block(Y, "Y")
        B = int(B) if B is not None else min(N, 256)
        ws = workspace if workspace is not None else self.workspace(min(B, N))
        Hh = torch.empty((N, N), dtype=torch.float64, device="cuda")
        self._check(load_library().chfsi_projected_hamiltonian_mixed(self._h, yp, ldy, N, B, int(n_oc), C.c_void_p(Hh.data_ptr()),
                                                                     C.c_void_p(ws.data_ptr()), _stream_ptr(stream)))
        return Hh

    def subspace_transform_mixed(self, Y, Z, Out=None, stream=None):
        """Out = SP[Y Z_od] + DP[Y Z_d] for a square Z (Z = L^-T gives the orthonormal basis Psi^o)."""
        import torch
        yp, ldy, N = self._block(Y, "Y")
        if Z.dim() != 2 or Z.shape[0] != N or Z.shape[1] != N or Z.dtype != torch.float64 or Z.stride(1) != 1 or not Z.is_cuda:
            raise ValueError("Z must be a [N, N] FP64 CUDA tensor with unit column stride")
        if Out is None:
            Out = torch.empty((self.n_dofs, N), dtype=torch.float64, device="cuda")
        op_, ldo, No = self._block(Out, "Out")
        if No != N:
            raise ValueError("Out must have N columns")
        self._check(load_library().chfsi_subspace_transform_mixed(self._h, yp, ldy, N, C.c_void_p(Z.data_ptr()),
                                                                  int(Z.stride(0)), op_, ldo, _stream_ptr(stream)))
        return Out

    def chebyshev_filter(self, X, m, a, b, a0, workspace=None, stream=None):
        """In place on the columns of X."""
        xp, ldx, B = self._block(X, "X")
        ws = workspace if workspace is not None else self.workspace(B)
        self._check(load_library().chfsi_chebyshev_filter(self._h, xp, ldx, B, int(m), float(a), float(b),
                                                          float(a0), C.c_void_p(ws.data_ptr()),
                                                          _stream_ptr(stream)))
        return X

    def chebyshev_filter_chunked(self, X, B, m, a, b, a0, workspace=None, stream=None):
        """In place on all N columns of X, filtered in sequential chunks of B columns."""
        xp, ldx, N = self._block(X, "X")
        B = min(int(B), N)
        ws = workspace if workspace is not None else self.workspace(B)
        self._check(load_library().chfsi_chebyshev_filter_chunked(self._h, xp, ldx, N, B, int(m), float(a),
                                                                  float(b), float(a0),
                                                                  C.c_void_p(ws.data_ptr()), _stream_ptr(stream)))
        return X

    def chebyshev_filter_host(self, X_host, B, m, a, b, a0):
        """End-to-end variant on a HOST block (NumPy array or CPU torch tensor, ideally pinned), in place."""
        import torch
        if isinstance(X_host, torch.Tensor):
            if X_host.is_cuda or X_host.dim() != 2 or X_host.stride(1) != 1 or X_host.dtype != self.dtype:
                raise TypeError("X_host: expected a 2-D CPU tensor of the operator's precision, vector index fastest")
            ptr, ld, N, rows = X_host.data_ptr(), X_host.stride(0), X_host.shape[1], X_host.shape[0]
        else:
            want = np.complex128 if self.kpoint else np.float64 if self.precision == 64 else np.float32
            if X_host.dtype != want or X_host.ndim != 2 or X_host.strides[1] != X_host.itemsize:
                raise TypeError("X_host: expected a 2-D array of the operator's precision, vector index fastest")
            ptr, ld, N, rows = X_host.ctypes.data, X_host.strides[0] // X_host.itemsize, X_host.shape[1], X_host.shape[0]
        if rows != self.n_dofs:
            raise ValueError("X_host: wrong number of rows")
        self._check(load_library().chfsi_chebyshev_filter_host(self._h, C.c_void_p(ptr), int(ld), int(N), int(B),
                                                               int(m), float(a), float(b), float(a0)))
        return X_host

    def launch_count(self) -> int:
        return int(load_library().chfsi_launch_count(self._h))

    def update_potential(self, veff_q, stream=None):
        """chfsi_update_potential: new V_eff samples [n_cells][(p+2)^3] (host array) on the same mesh/projectors."""
        v = np.ascontiguousarray(veff_q, dtype=np.float64)
        pot = _Potential(_np_ptr(v))
        self._check(load_library().chfsi_update_potential(self._h, C.byref(pot), _stream_ptr(stream)))

    def set_kernel_variant(self, variant: int):
        self._check(load_library().chfsi_set_kernel_variant(self._h, int(variant)))

    def set_rr_variant(self, variant: int):
        self._check(load_library().chfsi_set_rr_variant(self._h, int(variant)))

    def set_profiling(self, enabled: bool):
        self._check(load_library().chfsi_set_profiling(self._h, int(bool(enabled))))

    def get_profile(self) -> dict:
        pr = _Profile()
        self._check(load_library().chfsi_get_profile(self._h, C.byref(pr)))
        return {k: getattr(pr, k) for k, _ in _Profile._fields_}

    def close(self):
        if self._h is not None and _lib is not None:
            _lib.chfsi_destroy(self._h)
        self._h = None
        self._ws = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass
