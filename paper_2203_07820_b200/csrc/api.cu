// C ABI of libchfsi (include/chfsi.h): argument checking, operator construction, the Chebyshev host loop.
//
// The filter loop (Eq. 37, scaled form of ref. [86]) only computes the FP64 scalars
// sigma_k on the host and enqueues one fused "H~ apply + recurrence" launch sequence per degree on the caller's
// stream; it never synchronises.  Two blocks ping-pong: the caller's X and one workspace block W
//     k = 1 :  W <- (sigma_1/e)(H~ X - c X)
//     k = 2 :  X <- (2 sigma_2/e)(H~ W - c W) - sigma_1 sigma_2 X        (target holds Y_{k-2}, becomes Y_k)
//     ...
// and for odd m the result is copied from W back to X.
#include <cmath>
#include <cstdio>
#include <cstring>
#include <exception>
#include <new>

#include "common.h"

using namespace chfsi;

struct chfsi_op : public Op {};

namespace {

thread_local std::string g_create_error;

inline size_t align_up(size_t v, size_t a) { return (v + a - 1) / a * a; }

int fail(chfsi_op* op, int code, const std::string& msg) {
  if (op) op->err = msg; else g_create_error = msg;
  return code;
}
int cuda_fail(chfsi_op* op, cudaError_t e, const char* where) {
  return fail(op, e == cudaErrorMemoryAllocation ? CHFSI_ERR_OUT_OF_MEMORY : CHFSI_ERR_CUDA,
              std::string(where) + ": " + cudaGetErrorString(e));
}

template <typename U>
cudaError_t upload_vec(U** dst, const std::vector<U>& v, cudaStream_t st) {
  *dst = nullptr;
  size_t n = v.empty() ? 1 : v.size();
  cudaError_t e = cudaMalloc((void**)dst, n * sizeof(U));
  if (e != cudaSuccess) return e;
  if (!v.empty()) e = cudaMemcpyAsync(*dst, v.data(), v.size() * sizeof(U), cudaMemcpyHostToDevice, st);
  return e;
}

void free_op(chfsi_op* op) {
  if (!op) return;
  cudaFree(op->mat); cudaFree(op->mat_off); cudaFree(op->idx_off); cudaFree(op->ktot); cudaFree(op->gidx);
  cudaFree(op->color_cells); cudaFree(op->dep_ptr); cudaFree(op->dep_pos); cudaFree(op->all_cells); cudaFree(op->pc_cells); cudaFree(op->cell_proj_ptr);
  cudaFree(op->proj_ptr); cudaFree(op->proj_pcrow); cudaFree(op->seg_ptr); cudaFree(op->grow_dof); cudaFree(op->pcoef);
  cudaFree(op->grp_seg_ptr); cudaFree(op->proj_grp); cudaFree(op->proj_slot);
  cudaFree(op->rr_scratch); cudaFree(op->rr_flag); cudaFree(op->rr32[0]); cudaFree(op->rr32[1]); cudaFree(op->sf_coef); cudaFree(op->sf_sloc); cudaFree(op->crows);
  cudaFree(op->pcoef_im); cudaFree(op->seg_slot_proj); cudaFree(op->back_segs); cudaFree(op->veff_dev);
  for (int i = 0; i < 2; ++i) {
    cudaFree(op->host_stage[i]);
    if (op->host_done[i]) cudaEventDestroy(op->host_done[i]);
    if (op->host_st[i]) cudaStreamDestroy(op->host_st[i]);
  }
  cudaFree(op->host_ws);
  if (op->order_ev) cudaEventDestroy(op->order_ev);
  cudaFree(op->setup_verts); cudaFree(op->setup_pp); cudaFree(op->setup_phi); cudaFree(op->setup_gx); cudaFree(op->setup_gw); cudaFree(op->D); cudaFree(op->mass); cudaFree(op->diag0);
  for (cudaEvent_t e : op->prof_events) cudaEventDestroy(e);
  delete op;
}

struct WsLayout {
  size_t elt, block_off, p_off, pc_off, sync_off, sync_bytes, total;
  int64_t ldw;
};
WsLayout ws_layout(const Op* op, int64_t B) {
  WsLayout w;
  w.elt = op->precision == 64 ? 8 : 4;
  w.ldw = (B + 7) / 8 * 8;                                  // rows of the workspace block stay 32/64-byte aligned
  w.block_off = 0;
  w.p_off = align_up((size_t)op->n_dofs * w.ldw * w.elt, 256);
  w.pc_off = w.p_off + align_up((size_t)(op->n_proj + 1) * B * w.elt, 256);
  w.sync_off = w.pc_off + align_up((size_t)(op->n_pseg > 0 ? op->n_pseg : 1) * kProjGroup * B * sizeof(double), 256);
  // ticket counter (first 128 bytes) + one completion flag per (cell, 32-column tile): apply_kernels.cu, v2 kernel
  // (16-column tiles in the sum-factorised FP64 kernel)
  w.sync_bytes = align_up(128 + (size_t)op->n_cells * op->n_parts * (size_t)((B + 15) / 16) * sizeof(uint32_t), 256);
  w.total = w.sync_off + w.sync_bytes;
  return w;
}

int check_block_args(chfsi_op* op, const void* X, int64_t ldx, int64_t B, const void* ws) {
  if (!op) return CHFSI_ERR_BAD_ARGUMENT;
  if (!X) return fail(op, CHFSI_ERR_BAD_ARGUMENT, "NULL vector block");
  if (B < 1) return fail(op, CHFSI_ERR_BAD_ARGUMENT, "B < 1");
  if (B > (1 << 20)) return fail(op, CHFSI_ERR_BAD_ARGUMENT, "B too large");
  if (ldx < B) return fail(op, CHFSI_ERR_BAD_ARGUMENT, "ld < B");
  if (!ws) return fail(op, CHFSI_ERR_BAD_ARGUMENT, "NULL workspace");
  if ((uintptr_t)ws % 16 != 0) return fail(op, CHFSI_ERR_BAD_ARGUMENT, "workspace must be 16-byte aligned");
  return CHFSI_OK;
}

int filter_block(chfsi_op* op, void* X, int64_t ldx, int64_t B, int32_t m, double a, double b, double a0,
                 void* ws, cudaStream_t st) {
  const WsLayout w = ws_layout(op, B);
  char* base = reinterpret_cast<char*>(ws);
  void* W = base + w.block_off;
  ApplyArgs g;
  g.B = B; g.P = base + w.p_off; g.Pc = base + w.pc_off;
  g.sync = reinterpret_cast<unsigned long long*>(base + w.sync_off);
  cudaError_t cm = cudaMemsetAsync(g.sync, 0, w.sync_bytes, st);
  if (cm != cudaSuccess) return cuda_fail(op, cm, "chebyshev_filter memset");
  op->launches++;
  const double e = 0.5 * (b - a), c = 0.5 * (b + a);
  const double sigma1 = e / (a0 - c);
  double sigma = sigma1;
  void* cur = X; int64_t ldcur = ldx;      // Y_{k-1}
  void* tgt = W; int64_t ldtgt = w.ldw;    // Y_{k-2} -> Y_k
  // Scaled form of the recurrence for kernels that only add into the target block (ApplyArgs::accumulate): the blocks
  // hold W_k = s_k Y_k with s_0 = s_1 = 1 and s_k = -s_{k-2} / beta_k, so that
  //   Y_k = alpha_k (H~ - c) Y_{k-1} - beta_k Y_{k-2}   <=>   W_k = W_{k-2} + (s_k alpha_k / s_{k-1}) (H~ - c) W_{k-1},
  // and the result is W_m / s_m.  |s_k| = T_k(t0) / T_{k mod 2}(t0) (the unnormalised Chebyshev polynomials at
  // t0 = (a0 - c) / e): when that leaves the range of the storage type the three-term form is used instead.
  g.X = cur; g.ldx = ldcur; g.T = tgt; g.ldt = ldtgt;
  bool scaled = m >= 2 && apply_accumulates(op, g);
  if (scaled) {
    const double limit = op->precision == 64 ? 1e200 : 1e25;
    double s2 = 1.0, s1 = 1.0, sg = sigma1;
    for (int k = 2; k <= m && scaled; ++k) {
      const double sn = 1.0 / (2.0 / sigma1 - sg);
      const double sk = -s2 / (sg * sn);
      if (!(std::fabs(sk) < limit && std::fabs(sk) > 1.0 / limit)) scaled = false;
      s2 = s1; s1 = sk; sg = sn;
    }
  }
  if (op->kpoint && m >= 2 && !scaled)
    return fail(op, CHFSI_ERR_UNSUPPORTED, "k-point filter: block not aligned for the sum-factorised kernel, or T_m(t0) out of range");
  double s_km2 = 1.0, s_km1 = 1.0;         // s_{k-2}, s_{k-1}
  for (int k = 1; k <= m; ++k) {
    g.X = cur; g.ldx = ldcur; g.T = tgt; g.ldt = ldtgt; g.cshift = c; g.epoch = (uint32_t)k;
    g.accumulate = false;
    if (k == 1) { g.alpha = sigma1 / e; g.beta = 0.0; }
    else {
      const double sigma_new = 1.0 / (2.0 / sigma1 - sigma);
      g.alpha = 2.0 * sigma_new / e; g.beta = sigma * sigma_new; sigma = sigma_new;
      if (scaled) {
        const double s_k = -s_km2 / g.beta;
        g.alpha = s_k * g.alpha / s_km1; g.beta = 0.0; g.accumulate = true;
        s_km2 = s_km1; s_km1 = s_k;
      }
    }
    cudaError_t ce = launch_apply(op, g, st);
    if (ce != cudaSuccess) return cuda_fail(op, ce, "chebyshev_filter launch");
    std::swap(cur, tgt); std::swap(ldcur, ldtgt);
  }
  if (scaled) {     // X <- W_m / s_m (from the workspace block when m is odd, in place when m is even)
    cudaError_t ce = launch_scale_block(op, X, ldx, cur, ldcur, B, 1.0 / s_km1, st);
    if (ce != cudaSuccess) return cuda_fail(op, ce, "chebyshev_filter rescale");
  } else if (cur != X) {   // odd m: result sits in the workspace block
    cudaError_t ce = cudaMemcpy2DAsync(X, (size_t)ldx * w.elt, W, (size_t)w.ldw * w.elt, (size_t)B * w.elt,
                                       (size_t)op->n_dofs, cudaMemcpyDeviceToDevice, st);
    if (ce != cudaSuccess) return cuda_fail(op, ce, "chebyshev_filter copy-back");
    op->launches++;
  }
  return CHFSI_OK;
}

// One handle carries mutable state (the spectral shift on the matrix diagonals, scratch buffers, counters), so the
// device work of successive calls on one handle must not overlap.  Calls on DIFFERENT streams are therefore chained
// through an event: each call first makes its stream wait for the previous call's work on this handle.
cudaError_t order_enter(chfsi_op* op, cudaStream_t st) {
  if (op->order_valid && st != op->order_stream) return cudaStreamWaitEvent(st, op->order_ev, 0);
  return cudaSuccess;
}
cudaError_t order_leave(chfsi_op* op, cudaStream_t st) {
  if (!op->order_ev) {
    cudaError_t e = cudaEventCreateWithFlags(&op->order_ev, cudaEventDisableTiming);
    if (e != cudaSuccess) return e;
  }
  cudaError_t e = cudaEventRecord(op->order_ev, st);
  if (e == cudaSuccess) { op->order_stream = st; op->order_valid = true; }
  return e;
}

// Nothing throws across the ABI: every entry point runs its body inside API_TRY / API_CATCH.
#define API_TRY try {
#define API_CATCH(op_)                                                                                        \
  } catch (const std::bad_alloc&) { return fail(op_, CHFSI_ERR_OUT_OF_MEMORY, "host allocation failed"); }    \
    catch (const std::exception& ex_) { return fail(op_, CHFSI_ERR_CUDA, std::string("internal error: ") + ex_.what()); } \
    catch (...) { return fail(op_, CHFSI_ERR_CUDA, "internal error"); }

int check_filter_scalars(chfsi_op* op, int32_t m, double a, double b, double a0) {
  if (m < 1) return fail(op, CHFSI_ERR_BAD_ARGUMENT, "m < 1");
  if (!(a0 <= a && a < b) || !std::isfinite(a0) || !std::isfinite(b))
    return fail(op, CHFSI_ERR_BAD_ARGUMENT, "need finite a0 <= a < b");
  return CHFSI_OK;
}

}  // namespace

namespace {
// columns of the real block behind one column of the caller's block: 2 for the complex blocks of a k-point handle
inline int64_t col_width(const chfsi_op* op) { return op->kpoint ? 2 : 1; }

int create_impl(chfsi_op** out, const chfsi_mesh* mesh, const chfsi_potential* pot_in, const chfsi_nonlocal* nl,
                const chfsi_kpoint* kp, const double* dof_mass, int precision, int assembly, void* cuda_stream) {
  if (!out) return fail(nullptr, CHFSI_ERR_BAD_ARGUMENT, "out == NULL");
  *out = nullptr;
  if (!mesh || !pot_in || !mesh->cell_dofs || !mesh->cell_vertices || !pot_in->veff_q)
    return fail(nullptr, CHFSI_ERR_BAD_ARGUMENT, "NULL mesh / potential pointer");
  if (kp && (mesh->p > 6 || precision != 64))
    return fail(nullptr, CHFSI_ERR_UNSUPPORTED, "the k-point variant needs FE degree p <= 6 and precision 64");
  if (kp && !(std::isfinite(kp->k[0]) && std::isfinite(kp->k[1]) && std::isfinite(kp->k[2])))
    return fail(nullptr, CHFSI_ERR_BAD_ARGUMENT, "non-finite k vector");
  if (mesh->p < 1 || mesh->p > 8) return fail(nullptr, CHFSI_ERR_UNSUPPORTED, "FE degree p must be in 1..8");
  if (precision != 64 && precision != 32) return fail(nullptr, CHFSI_ERR_UNSUPPORTED, "precision must be 64 or 32");
  if (assembly != 0 && assembly != 1) return fail(nullptr, CHFSI_ERR_BAD_ARGUMENT, "assembly must be 0 or 1");
  if (mesh->n_cells < 1 || mesh->n_dofs < 1 || mesh->n_cells > INT32_MAX / 2 || mesh->n_dofs > INT32_MAX / 2)
    return fail(nullptr, CHFSI_ERR_BAD_ARGUMENT, "n_cells / n_dofs out of range");
  const bool has_nl = nl && nl->n_proj > 0;
  if (has_nl && (!nl->D || !nl->proj_cell_ptr || !nl->proj_cell_idx || !nl->chi_q))
    return fail(nullptr, CHFSI_ERR_BAD_ARGUMENT, "NULL projector pointer");

  int ndev = 0;
  cudaError_t ce = cudaGetDeviceCount(&ndev);
  if (ce != cudaSuccess || ndev == 0)
    return fail(nullptr, CHFSI_ERR_CUDA, std::string("no CUDA device (there is no CPU fallback): ") +
                                             (ce != cudaSuccess ? cudaGetErrorString(ce) : "device count 0"));
  cudaStream_t st = reinterpret_cast<cudaStream_t>(cuda_stream);

  if (kp && has_nl && !kp->chi_q_im) return fail(nullptr, CHFSI_ERR_BAD_ARGUMENT, "NULL chi_q_im with projectors");
  chfsi_op* op = new (std::nothrow) chfsi_op();
  if (!op) return fail(nullptr, CHFSI_ERR_OUT_OF_MEMORY, "host allocation failed");
  try {
  // k-point variant: the term 1/2 |k|^2 of Eq. 30 joins V_eff at the Gauss points
  std::vector<double> veff_k;
  chfsi_potential pot_k = *pot_in;
  const chfsi_potential* pot = pot_in;
  if (kp) {
    op->kpoint = true;
    for (int i = 0; i < 3; ++i) op->kvec[i] = kp->k[i];
    const int64_t nq = (int64_t)(mesh->p + 2) * (mesh->p + 2) * (mesh->p + 2);
    const double half_k2 = 0.5 * (kp->k[0] * kp->k[0] + kp->k[1] * kp->k[1] + kp->k[2] * kp->k[2]);
    veff_k.resize((size_t)(mesh->n_cells * nq));
    for (size_t i = 0; i < veff_k.size(); ++i) veff_k[i] = pot_in->veff_q[i] + half_k2;
    pot_k.veff_q = veff_k.data();
    pot = &pot_k;
  }
  op->p = mesh->p; op->n1 = mesh->p + 1; op->nq1 = mesh->p + 2;
  op->m_cell = op->n1 * op->n1 * op->n1; op->n_q = op->nq1 * op->nq1 * op->nq1;
  op->mpad = (op->m_cell + 7) / 8 * 8;
  // leading dimension of the cell matrices = their shared-memory row pitch: the four k-rows of an mma A fragment
  // must fall into different bank groups.  FP64: LDA mod 16 in {4, 12}; FP32: LDA mod 32 in {8, 24}.
  {
    const int n_mtiles = op->mpad / 8;
    op->n_parts = (n_mtiles + kMaxPartMTiles - 1) / kMaxPartMTiles;
    op->mw = 8 * ((n_mtiles + op->n_parts - 1) / op->n_parts);
  }
  op->lda = precision == 64 ? op->mw + 4 : op->mw + (op->mw % 16 == 0 ? 8 : 0);
  op->precision = precision; op->assembly = assembly;
  op->n_cells = mesh->n_cells; op->n_dofs = mesh->n_dofs; op->n_proj = has_nl ? nl->n_proj : 0;

  Tables1D tab;
  build_tables(op->p, &tab);
  HostPlan plan;
  std::string msg = analyse_mesh(*mesh, has_nl ? nl : nullptr, tab, op->lda, op->n_parts, &plan);
  if (!msg.empty()) { free_op(op); return fail(nullptr, CHFSI_ERR_BAD_MESH, msg); }
  if (dof_mass) {   // a part of a larger mesh: the diagonal mass of the WHOLE mesh at these dofs (chfsi_create_part)
    for (int64_t g = 0; g < mesh->n_dofs; ++g)
      if (!(dof_mass[g] > 0.0) || !std::isfinite(dof_mass[g])) {
        free_op(op);
        return fail(nullptr, CHFSI_ERR_BAD_ARGUMENT, "dof_mass must be positive and finite");
      }
    plan.mass.assign(dof_mass, dof_mass + mesh->n_dofs);
  }

  op->n_colors = plan.n_colors; op->color_ptr = plan.color_ptr;
  op->nnz_cp = (int64_t)plan.cell_proj_idx.size();
  op->n_pc_cells = (int64_t)plan.pc_cells.size();
  op->max_ktot = 0;
  for (int32_t k : plan.ktot) op->max_ktot = std::max(op->max_ktot, (int)k);
  op->mat_elems = plan.mat_off[op->n_cells];

#define CKC(x, what) do { ce = (x); if (ce != cudaSuccess) { int rc_ = cuda_fail(nullptr, ce, what); free_op(op); return rc_; } } while (0)
  const size_t elt = precision == 64 ? 8 : 4;
  CKC(cudaMalloc(&op->mat, (size_t)op->mat_elems * elt), "cudaMalloc(cell matrices)");
  CKC(upload_vec(&op->mat_off, plan.mat_off, st), "upload");
  CKC(upload_vec(&op->idx_off, plan.idx_off, st), "upload");
  CKC(upload_vec(&op->ktot, plan.ktot, st), "upload");
  CKC(upload_vec(&op->gidx, plan.gidx, st), "upload");
  CKC(upload_vec(&op->color_cells, plan.color_cells, st), "upload");
  CKC(upload_vec(&op->dep_ptr, plan.dep_ptr, st), "upload");
  CKC(upload_vec(&op->dep_pos, plan.dep_pos, st), "upload");
  {
    int dev = 0;
    CKC(cudaGetDevice(&dev), "cudaGetDevice");
    CKC(cudaDeviceGetAttribute(&op->n_sm, cudaDevAttrMultiProcessorCount, dev), "SM count");
  }
  {
    std::vector<int32_t> all(op->n_cells);
    for (int64_t c = 0; c < op->n_cells; ++c) all[c] = (int32_t)c;
    CKC(upload_vec(&op->all_cells, all, st), "upload");
    CKC(cudaStreamSynchronize(st), "sync");
  }
  CKC(upload_vec(&op->pc_cells, plan.pc_cells, st), "upload");
  CKC(upload_vec(&op->cell_proj_ptr, plan.cell_proj_ptr, st), "upload");
  CKC(upload_vec(&op->proj_ptr, plan.proj_ptr, st), "upload");
  CKC(upload_vec(&op->proj_pcrow, plan.proj_pcrow, st), "upload");
  CKC(upload_vec(&op->seg_ptr, plan.seg_ptr, st), "upload");
  CKC(upload_vec(&op->grow_dof, plan.grow_dof, st), "upload");
  CKC(upload_vec(&op->grp_seg_ptr, plan.grp_seg_ptr, st), "upload");
  CKC(upload_vec(&op->proj_grp, plan.proj_grp, st), "upload");
  CKC(upload_vec(&op->proj_slot, plan.proj_slot, st), "upload");
  {
    std::vector<double> D(has_nl ? nl->D : nullptr, has_nl ? nl->D + nl->n_proj : nullptr);
    CKC(upload_vec(&op->D, D, st), "upload");
    CKC(cudaStreamSynchronize(st), "sync");
  }
  CKC(upload_vec(&op->mass, plan.mass, st), "upload");
  bool bad_jac = false;
  CKC(build_cell_matrices(op, plan, tab, *mesh, *pot, has_nl ? nl : nullptr, st, &bad_jac), "cell-matrix setup");
  if (bad_jac) { free_op(op); return fail(nullptr, CHFSI_ERR_BAD_MESH, "non-positive Jacobian at a quadrature point"); }
  CKC(assemble_projector_rows(op, plan, *mesh, st), "projector-row assembly");
  CKC(cudaMalloc((void**)&op->diag0, (size_t)op->n_cells * op->m_cell * sizeof(double)), "cudaMalloc(diagonal)");
  CKC(capture_diagonal(op, st), "diagonal capture");
  CKC(init_apply_kernels(op), "kernel attribute setup");
  CKC(init_sf_variant(op, tab, st), "sum-factorised variant setup");
  if (op->sf_ok) CKC(build_sf_fields(op, pot->veff_q, st), "quadrature-point fields");
  if (kp) {
    if (!op->sf_ok) {
      free_op(op);
      return fail(nullptr, CHFSI_ERR_UNSUPPORTED, "the k-point variant needs the sum-factorised kernel");
    }
    if (has_nl && op->nnz_cp > 0) {   // imaginary parts of the projector coefficients: the same path on chi_q_im
      CKC(build_cell_projectors(op, plan, kp->chi_q_im, st), "cell projectors (imaginary parts)");
      CKC(assemble_projector_rows_imag(op, plan, *mesh, st), "projector-row assembly (imaginary parts)");
    }
  }
  CKC(cudaStreamSynchronize(st), "sync");
#undef CKC
  } catch (const std::bad_alloc&) {
    free_op(op);
    return fail(nullptr, CHFSI_ERR_OUT_OF_MEMORY, "host allocation failed in chfsi_create");
  } catch (...) {
    free_op(op);
    return fail(nullptr, CHFSI_ERR_CUDA, "internal error in chfsi_create");
  }
  *out = op;
  return CHFSI_OK;
}

}  // namespace

extern "C" {

int chfsi_create(chfsi_op** out, const chfsi_mesh* mesh, const chfsi_potential* pot, const chfsi_nonlocal* nl,
                 int precision, int assembly, void* cuda_stream) {
  return create_impl(out, mesh, pot, nl, nullptr, nullptr, precision, assembly, cuda_stream);
}

int chfsi_create_k(chfsi_op** out, const chfsi_mesh* mesh, const chfsi_potential* pot, const chfsi_nonlocal* nl,
                   const chfsi_kpoint* kpoint, int assembly, void* cuda_stream) {
  if (!kpoint) return fail(nullptr, CHFSI_ERR_BAD_ARGUMENT, "kpoint == NULL");
  return create_impl(out, mesh, pot, nl, kpoint, nullptr, 64, assembly, cuda_stream);
}

int chfsi_create_part(chfsi_op** out, const chfsi_mesh* mesh, const chfsi_potential* pot, const chfsi_nonlocal* nl,
                      const double* dof_mass, int precision, int assembly, void* cuda_stream) {
  if (!dof_mass) return fail(nullptr, CHFSI_ERR_BAD_ARGUMENT, "dof_mass == NULL");
  return create_impl(out, mesh, pot, nl, nullptr, dof_mass, precision, assembly, cuda_stream);
}

int chfsi_mesh_mass(const chfsi_mesh* mesh, double* mass_host) {
  if (!mesh || !mass_host || !mesh->cell_dofs || !mesh->cell_vertices) return CHFSI_ERR_BAD_ARGUMENT;
  if (mesh->p < 1 || mesh->p > 8) return CHFSI_ERR_UNSUPPORTED;
  if (mesh->n_cells < 1 || mesh->n_dofs < 1) return CHFSI_ERR_BAD_ARGUMENT;
  try {
    Tables1D tab;
    build_tables(mesh->p, &tab);
    std::vector<double> m;
    const std::string msg = mesh_mass(*mesh, tab, &m);
    if (!msg.empty()) { g_create_error = msg; return CHFSI_ERR_BAD_MESH; }
    std::copy(m.begin(), m.end(), mass_host);
    return CHFSI_OK;
  } catch (...) {
    return CHFSI_ERR_OUT_OF_MEMORY;
  }
}

int chfsi_destroy(chfsi_op* op) {
  if (!op) return CHFSI_ERR_BAD_ARGUMENT;
  free_op(op);
  return CHFSI_OK;
}

int chfsi_update_potential(chfsi_op* op, const chfsi_potential* pot, void* cuda_stream) {
  if (!op) return CHFSI_ERR_BAD_ARGUMENT;
  if (!pot || !pot->veff_q) return fail(op, CHFSI_ERR_BAD_ARGUMENT, "NULL potential pointer");
  API_TRY
  cudaStream_t st = reinterpret_cast<cudaStream_t>(cuda_stream);
  std::vector<double> veff_k;
  const double* veff_q = pot->veff_q;
  if (op->kpoint) {   // V_eff + 1/2 |k|^2 (Eq. 30), as at creation
    const double half_k2 = 0.5 * (op->kvec[0] * op->kvec[0] + op->kvec[1] * op->kvec[1] + op->kvec[2] * op->kvec[2]);
    veff_k.resize((size_t)(op->n_cells * op->n_q));
    for (size_t i = 0; i < veff_k.size(); ++i) veff_k[i] = pot->veff_q[i] + half_k2;
    veff_q = veff_k.data();
  }
  cudaError_t ce = order_enter(op, st);
  if (ce != cudaSuccess) return cuda_fail(op, ce, "update_potential");
  if (op->sf_ok) {
    // the default kernel is sum-factorised: its operator data are the quadrature-point fields, rebuilt in one small kernel
    // from the samples; the dense cell matrices (other kernel variants) follow lazily from the device copy of the samples
    const size_t bytes = (size_t)op->n_cells * op->n_q * sizeof(double);
    if (!op->veff_dev) ce = cudaMalloc((void**)&op->veff_dev, bytes);
    if (ce == cudaSuccess) ce = cudaMemcpyAsync(op->veff_dev, veff_q, bytes, cudaMemcpyHostToDevice, st);
    if (ce == cudaSuccess) ce = build_sf_fields_dev(op, op->veff_dev, st);
    if (ce == cudaSuccess) ce = cudaStreamSynchronize(st);      // veff_q (caller's / veff_k) may go away after the call
    if (ce != cudaSuccess) return cuda_fail(op, ce, "update_potential (quadrature-point fields)");
    op->dense_stale = !op->kpoint;
    op->launches += 1;
  } else {
    ce = rebuild_local_matrices(op, veff_q, st);
    if (ce != cudaSuccess) return cuda_fail(op, ce, "update_potential (cell matrices)");
    ce = capture_diagonal(op, st);      // new unshifted diagonals; the spectral shift of the last filter is gone
    if (ce == cudaSuccess) ce = cudaStreamSynchronize(st);
    if (ce != cudaSuccess) return cuda_fail(op, ce, "update_potential (diagonal)");
    op->launches += 2;
  }
  op->order_valid = false;             // the stream was synchronised: nothing of this handle is in flight
  return CHFSI_OK;
  API_CATCH(op)
}

int chfsi_get_info(const chfsi_op* op, chfsi_info* info) {
  if (!op || !info) return CHFSI_ERR_BAD_ARGUMENT;
  info->p = op->p; info->m_cell = op->m_cell; info->n_q = op->n_q; info->precision = op->precision;
  info->assembly = op->assembly; info->n_colors = op->n_colors;
  info->n_cells = op->n_cells; info->n_dofs = op->n_dofs; info->n_proj = op->n_proj;
  info->nnz_cell_proj = op->nnz_cp; info->cells_with_proj = op->n_pc_cells;
  info->flops_per_vector_apply = (double)op->n_cells * 2.0 * op->m_cell * op->m_cell +
                                 4.0 * op->m_cell * (double)op->nnz_cp + 7.0 * (double)op->n_dofs;
  info->matrix_bytes = op->mat_elems * (op->precision == 64 ? 8 : 4);
  info->sf_flops_per_vector_apply = 0.0; info->sf_field_bytes = 0;
  if (op->sf_ok) {
    // executed work of k_apply_sf per (cell, column): DMMAs of the eight MMA stages, the in-lane DFMA stages, the
    // Gauss-point stage, the scalings; per cell with projectors the k = 8 MMAs of the assembly (apply_sf.cuh)
    const double n1 = op->n1, nq1 = op->nq1;
    const double dmma = 8.0 * n1 + 8.0 * nq1;
    const double lane_flops = 2.0 * (4.0 * n1 * nq1 + 4.0 * nq1 * nq1) + 34.0 * nq1 + 10.0 * n1;
    const double per_cell_col = dmma * 512.0 + 32.0 * lane_flops;
    const double proj_per_cell_col = 2.0 * ((op->m_cell + 7) / 8) * 512.0 / 8.0;
    info->sf_flops_per_vector_apply = (double)op->n_cells * per_cell_col + (double)op->n_pc_cells * proj_per_cell_col +
                                      4.0 * (double)op->n_cells * op->m_cell;
    info->sf_field_bytes = (int64_t)op->n_cells * (op->nq1 * 7 * 64 + op->mpad) * 8;
  }
  return CHFSI_OK;
}

int chfsi_workspace_bytes(const chfsi_op* op, int64_t B, size_t* bytes) {
  if (!op || !bytes || B < 1) return CHFSI_ERR_BAD_ARGUMENT;
  *bytes = ws_layout(op, B * col_width(op)).total;
  return CHFSI_OK;
}

int chfsi_mass_diag(const chfsi_op* op, double* M_dev, void* cuda_stream) {
  if (!op || !M_dev) return CHFSI_ERR_BAD_ARGUMENT;
  cudaError_t ce = cudaMemcpyAsync(M_dev, op->mass, (size_t)op->n_dofs * sizeof(double), cudaMemcpyDeviceToDevice,
                                   reinterpret_cast<cudaStream_t>(cuda_stream));
  return ce == cudaSuccess ? CHFSI_OK : CHFSI_ERR_CUDA;
}

int chfsi_apply_H(chfsi_op* op, const void* X_dev, int64_t ldx, void* Y_dev, int64_t ldy, int64_t B,
                  void* workspace_dev, void* cuda_stream) {
  if (op) { ldx *= col_width(op); ldy *= col_width(op); B *= col_width(op); }    // complex columns = pairs of real columns
  int rc = check_block_args(op, X_dev, ldx, B, workspace_dev);
  if (rc) return rc;
  if (!Y_dev) return fail(op, CHFSI_ERR_BAD_ARGUMENT, "NULL output block");
  if (ldy < B) return fail(op, CHFSI_ERR_BAD_ARGUMENT, "ldy < B");
  if (X_dev == Y_dev) return fail(op, CHFSI_ERR_BAD_ARGUMENT, "X and Y must not overlap");
  API_TRY
  cudaStream_t st = reinterpret_cast<cudaStream_t>(cuda_stream);
  const WsLayout w = ws_layout(op, B);
  char* base = reinterpret_cast<char*>(workspace_dev);
  ApplyArgs g;
  g.X = X_dev; g.ldx = ldx; g.T = Y_dev; g.ldt = ldy; g.B = B;
  g.alpha = 1.0; g.beta = 0.0; g.cshift = 0.0;
  g.P = base + w.p_off; g.Pc = base + w.pc_off;
  g.sync = reinterpret_cast<unsigned long long*>(base + w.sync_off); g.epoch = 1;
  cudaError_t ce = order_enter(op, st);
  if (ce == cudaSuccess) ce = cudaMemsetAsync(g.sync, 0, w.sync_bytes, st);
  if (ce != cudaSuccess) return cuda_fail(op, ce, "apply_H memset");
  op->launches++;
  ce = launch_apply(op, g, st);
  if (ce == cudaSuccess) ce = order_leave(op, st);
  if (ce != cudaSuccess) return cuda_fail(op, ce, "apply_H launch");
  return CHFSI_OK;
  API_CATCH(op)
}

namespace {
// chfsi_apply_H in phases (ApplyArgs::phase): the projector coefficients of this operator's cells, or H~X with given ones
int apply_phase(chfsi_op* op, const void* X_dev, int64_t ldx, void* Y_dev, int64_t ldy, int64_t B, void* P_dev, int phase,
                void* workspace_dev, void* cuda_stream, double alpha = 1.0, double cshift = 0.0, bool accumulate = false,
                int* query = nullptr) {
  int rc = check_block_args(op, X_dev, ldx, B, workspace_dev);
  if (rc) return rc;
  if (op->kpoint) return fail(op, CHFSI_ERR_UNSUPPORTED, "phased application of a k-point handle");
  if (op->n_proj > 0 && !P_dev) return fail(op, CHFSI_ERR_BAD_ARGUMENT, "NULL coefficient block");
  if (phase == 2) {
    if (!Y_dev) return fail(op, CHFSI_ERR_BAD_ARGUMENT, "NULL output block");
    if (ldy < B) return fail(op, CHFSI_ERR_BAD_ARGUMENT, "ldy < B");
    if (X_dev == Y_dev) return fail(op, CHFSI_ERR_BAD_ARGUMENT, "X and Y must not overlap");
  }
  API_TRY
  cudaStream_t st = reinterpret_cast<cudaStream_t>(cuda_stream);
  const WsLayout w = ws_layout(op, B);
  char* base = reinterpret_cast<char*>(workspace_dev);
  ApplyArgs g;
  g.X = X_dev; g.ldx = ldx; g.T = phase == 2 ? Y_dev : const_cast<void*>(X_dev); g.ldt = phase == 2 ? ldy : ldx; g.B = B;
  g.alpha = alpha; g.beta = 0.0; g.cshift = cshift; g.phase = phase; g.accumulate = accumulate;
  g.P = base + w.p_off; g.Pc = base + w.pc_off;
  g.sync = reinterpret_cast<unsigned long long*>(base + w.sync_off); g.epoch = 1;
  if (query) { *query = apply_accumulates(op, g) ? 1 : 0; return CHFSI_OK; }
  if (accumulate && !apply_accumulates(op, g))
    return fail(op, CHFSI_ERR_UNSUPPORTED, "accumulating application: needs the sum-factorised kernel (p <= 6, variant 0 or 6) and aligned blocks");
  const size_t p_bytes = (size_t)op->n_proj * B * w.elt;
  cudaError_t ce = order_enter(op, st);
  if (ce == cudaSuccess) ce = cudaMemsetAsync(g.sync, 0, w.sync_bytes, st);
  if (ce == cudaSuccess && phase == 2) {   // rows 0 .. n_proj-1 from the caller, the all-zero row n_proj behind them
    if (p_bytes) ce = cudaMemcpyAsync(g.P, P_dev, p_bytes, cudaMemcpyDeviceToDevice, st);
    if (ce == cudaSuccess) ce = cudaMemsetAsync(reinterpret_cast<char*>(g.P) + p_bytes, 0, (size_t)B * w.elt, st);
  }
  if (ce != cudaSuccess) return cuda_fail(op, ce, "phased apply_H setup");
  op->launches++;
  ce = launch_apply(op, g, st);
  if (ce == cudaSuccess && phase == 1 && p_bytes) ce = cudaMemcpyAsync(P_dev, g.P, p_bytes, cudaMemcpyDeviceToDevice, st);
  if (ce == cudaSuccess) ce = order_leave(op, st);
  if (ce != cudaSuccess) return cuda_fail(op, ce, "phased apply_H launch");
  return CHFSI_OK;
  API_CATCH(op)
}
}  // namespace

int chfsi_projector_coefficients(chfsi_op* op, const void* X_dev, int64_t ldx, int64_t B, void* P_dev, void* workspace_dev,
                                 void* cuda_stream) {
  return apply_phase(op, X_dev, ldx, nullptr, 0, B, P_dev, 1, workspace_dev, cuda_stream);
}

int chfsi_apply_H_with_coefficients(chfsi_op* op, const void* X_dev, int64_t ldx, void* Y_dev, int64_t ldy, int64_t B,
                                    const void* P_dev, void* workspace_dev, void* cuda_stream) {
  return apply_phase(op, X_dev, ldx, Y_dev, ldy, B, const_cast<void*>(P_dev), 2, workspace_dev, cuda_stream);
}

int chfsi_apply_shifted_with_coefficients(chfsi_op* op, const void* X_dev, int64_t ldx, void* T_dev, int64_t ldt, int64_t B,
                                          double alpha, double c, int accumulate, const void* P_dev, void* workspace_dev,
                                          void* cuda_stream) {
  if (op && !(std::isfinite(alpha) && std::isfinite(c))) return fail(op, CHFSI_ERR_BAD_ARGUMENT, "alpha, c must be finite");
  return apply_phase(op, X_dev, ldx, T_dev, ldt, B, const_cast<void*>(P_dev), 2, workspace_dev, cuda_stream, alpha, c, accumulate != 0);
}

int chfsi_accumulate_supported(chfsi_op* op, const void* X_dev, int64_t ldx, const void* T_dev, int64_t ldt, int64_t B,
                               void* workspace_dev, int* supported) {
  if (op && !supported) return fail(op, CHFSI_ERR_BAD_ARGUMENT, "NULL result pointer");
  int dummy = 0;   // P_dev is not dereferenced by the query
  return apply_phase(op, X_dev, ldx, const_cast<void*>(T_dev), ldt, B, &dummy, 2, workspace_dev, nullptr, 1.0, 0.0, true, supported);
}

int chfsi_recurrence_update(chfsi_op* op, const void* HX_dev, int64_t ldh, const void* X_dev, int64_t ldx, void* T_dev,
                            int64_t ldt, int64_t B, double alpha, double beta, double c, void* cuda_stream) {
  if (!op) return CHFSI_ERR_BAD_ARGUMENT;
  if (!HX_dev || !X_dev || !T_dev) return fail(op, CHFSI_ERR_BAD_ARGUMENT, "NULL block");
  if (B < 1 || ldh < B || ldx < B || ldt < B) return fail(op, CHFSI_ERR_BAD_ARGUMENT, "need B >= 1 and ld >= B");
  if (op->kpoint) return fail(op, CHFSI_ERR_UNSUPPORTED, "recurrence_update on a k-point handle");
  API_TRY
  cudaStream_t st = reinterpret_cast<cudaStream_t>(cuda_stream);
  cudaError_t ce = order_enter(op, st);
  if (ce == cudaSuccess) ce = launch_recurrence(op, HX_dev, ldh, X_dev, ldx, T_dev, ldt, B, alpha, beta, c, st);
  if (ce == cudaSuccess) ce = order_leave(op, st);
  return ce == cudaSuccess ? CHFSI_OK : cuda_fail(op, ce, "recurrence_update");
  API_CATCH(op)
}

namespace {
int pack_rows(chfsi_op* op, const void* X_dev, int64_t ldx, int64_t B, const int32_t* rows_dev, const int32_t* slots_dev,
              int64_t n_rows, void* buf_dev, int buf_precision, bool unpack, void* cuda_stream) {
  if (!op) return CHFSI_ERR_BAD_ARGUMENT;
  if (n_rows < 0 || B < 1 || ldx < B) return fail(op, CHFSI_ERR_BAD_ARGUMENT, "need n_rows >= 0, B >= 1, ld >= B");
  if (n_rows > 0 && (!X_dev || !rows_dev || !buf_dev)) return fail(op, CHFSI_ERR_BAD_ARGUMENT, "NULL pointer");
  if (buf_precision != op->precision && buf_precision != 32)
    return fail(op, CHFSI_ERR_BAD_ARGUMENT, "buf_precision must be the operator's precision or 32");
  if (op->kpoint) return fail(op, CHFSI_ERR_UNSUPPORTED, "pack / unpack on a k-point handle");
  API_TRY
  cudaStream_t st = reinterpret_cast<cudaStream_t>(cuda_stream);
  cudaError_t ce = order_enter(op, st);
  if (ce == cudaSuccess) ce = launch_pack_rows(op, X_dev, ldx, B, rows_dev, slots_dev, n_rows, buf_dev, buf_precision, unpack, st);
  if (ce == cudaSuccess) ce = order_leave(op, st);
  return ce == cudaSuccess ? CHFSI_OK : cuda_fail(op, ce, unpack ? "unpack_rows" : "pack_rows");
  API_CATCH(op)
}
}  // namespace

int chfsi_pack_rows(chfsi_op* op, const void* X_dev, int64_t ldx, int64_t B, const int32_t* rows_dev, const int32_t* slots_dev,
                    int64_t n_rows, void* buf_dev, int buf_precision, void* cuda_stream) {
  return pack_rows(op, X_dev, ldx, B, rows_dev, slots_dev, n_rows, buf_dev, buf_precision, false, cuda_stream);
}

int chfsi_unpack_rows(chfsi_op* op, const void* buf_dev, int buf_precision, const int32_t* rows_dev, const int32_t* slots_dev,
                      int64_t n_rows, void* X_dev, int64_t ldx, int64_t B, void* cuda_stream) {
  return pack_rows(op, X_dev, ldx, B, rows_dev, slots_dev, n_rows, const_cast<void*>(buf_dev), buf_precision, true, cuda_stream);
}

namespace {
int rows_delta(chfsi_op* op, void* T_dev, int64_t ldt, const void* base_dev, const void* X_dev, int64_t ldx, const uint8_t* owner_dev,
               double corr, int64_t B, const int32_t* rows_dev, const int32_t* slots_dev, int64_t n_rows, void* buf_dev,
               int buf_precision, bool unpack, void* cuda_stream) {
  if (!op) return CHFSI_ERR_BAD_ARGUMENT;
  if (n_rows < 0 || B < 1 || ldt < B) return fail(op, CHFSI_ERR_BAD_ARGUMENT, "need n_rows >= 0, B >= 1, ld >= B");
  if (n_rows > 0 && (!T_dev || !rows_dev || !buf_dev)) return fail(op, CHFSI_ERR_BAD_ARGUMENT, "NULL pointer");
  if (n_rows > 0 && !unpack && (!X_dev || !owner_dev || ldx < B || !std::isfinite(corr)))
    return fail(op, CHFSI_ERR_BAD_ARGUMENT, "pack_rows_delta: need X (ldx >= B), the owner flags and a finite correction factor");
  if (buf_precision != op->precision && buf_precision != 32)
    return fail(op, CHFSI_ERR_BAD_ARGUMENT, "buf_precision must be the operator's precision or 32");
  if (op->kpoint) return fail(op, CHFSI_ERR_UNSUPPORTED, "pack / unpack on a k-point handle");
  API_TRY
  cudaStream_t st = reinterpret_cast<cudaStream_t>(cuda_stream);
  cudaError_t ce = order_enter(op, st);
  if (ce == cudaSuccess)
    ce = launch_rows_delta(op, T_dev, ldt, base_dev, X_dev, ldx, owner_dev, corr, B, rows_dev, slots_dev, n_rows, buf_dev,
                           buf_precision, unpack, st);
  if (ce == cudaSuccess) ce = order_leave(op, st);
  return ce == cudaSuccess ? CHFSI_OK : cuda_fail(op, ce, unpack ? "unpack_rows_sum" : "pack_rows_delta");
  API_CATCH(op)
}
}  // namespace

int chfsi_pack_rows_delta(chfsi_op* op, const void* T_dev, int64_t ldt, const void* base_dev, const void* X_dev, int64_t ldx,
                          const uint8_t* owner_dev, double corr, int64_t B, const int32_t* rows_dev, const int32_t* slots_dev,
                          int64_t n_rows, void* buf_dev, int buf_precision, void* cuda_stream) {
  return rows_delta(op, const_cast<void*>(T_dev), ldt, base_dev, X_dev, ldx, owner_dev, corr, B, rows_dev, slots_dev, n_rows, buf_dev,
                    buf_precision, false, cuda_stream);
}

int chfsi_unpack_rows_sum(chfsi_op* op, const void* buf_dev, int buf_precision, const void* base_dev, const int32_t* rows_dev,
                          const int32_t* slots_dev, int64_t n_rows, void* T_dev, int64_t ldt, int64_t B, void* cuda_stream) {
  return rows_delta(op, T_dev, ldt, base_dev, nullptr, 0, nullptr, 0.0, B, rows_dev, slots_dev, n_rows, const_cast<void*>(buf_dev),
                    buf_precision, true, cuda_stream);
}

int chfsi_chebyshev_filter(chfsi_op* op, void* X_dev, int64_t ldx, int64_t B, int32_t m, double a, double b,
                           double a0, void* workspace_dev, void* cuda_stream) {
  if (op) { ldx *= col_width(op); B *= col_width(op); }
  int rc = check_block_args(op, X_dev, ldx, B, workspace_dev);
  if (rc) return rc;
  if ((rc = check_filter_scalars(op, m, a, b, a0))) return rc;
  API_TRY
  cudaStream_t st = reinterpret_cast<cudaStream_t>(cuda_stream);
  cudaError_t ce = order_enter(op, st);
  if (ce != cudaSuccess) return cuda_fail(op, ce, "chebyshev_filter");
  rc = filter_block(op, X_dev, ldx, B, m, a, b, a0, workspace_dev, st);
  if (rc) return rc;
  ce = order_leave(op, st);
  return ce == cudaSuccess ? CHFSI_OK : cuda_fail(op, ce, "chebyshev_filter");
  API_CATCH(op)
}

int chfsi_chebyshev_filter_chunked(chfsi_op* op, void* X_dev, int64_t ldx, int64_t N, int64_t B, int32_t m,
                                   double a, double b, double a0, void* workspace_dev, void* cuda_stream) {
  if (op) { ldx *= col_width(op); B *= col_width(op); N *= col_width(op); }
  int rc = check_block_args(op, X_dev, ldx, B, workspace_dev);
  if (rc) return rc;
  if (N < 1 || ldx < N) return fail(op, CHFSI_ERR_BAD_ARGUMENT, "need 1 <= N <= ld");
  if ((rc = check_filter_scalars(op, m, a, b, a0))) return rc;
  API_TRY
  const size_t elt = op->precision == 64 ? 8 : 4;
  cudaStream_t st = reinterpret_cast<cudaStream_t>(cuda_stream);
  cudaError_t ce = order_enter(op, st);
  if (ce != cudaSuccess) return cuda_fail(op, ce, "chebyshev_filter_chunked");
  for (int64_t j0 = 0; j0 < N; j0 += B) {
    const int64_t bw = std::min(B, N - j0);
    rc = filter_block(op, reinterpret_cast<char*>(X_dev) + (size_t)j0 * elt, ldx, bw, m, a, b, a0, workspace_dev, st);
    if (rc) return rc;
  }
  ce = order_leave(op, st);
  return ce == cudaSuccess ? CHFSI_OK : cuda_fail(op, ce, "chebyshev_filter_chunked");
  API_CATCH(op)
}

int chfsi_chebyshev_filter_host(chfsi_op* op, void* X_host, int64_t ldx, int64_t N, int64_t B, int32_t m, double a,
                                double b, double a0) {
  if (!op) return CHFSI_ERR_BAD_ARGUMENT;
  if (!X_host) return fail(op, CHFSI_ERR_BAD_ARGUMENT, "NULL host block");
  ldx *= col_width(op); N *= col_width(op); B *= col_width(op);
  if (B < 1 || N < 1 || ldx < N) return fail(op, CHFSI_ERR_BAD_ARGUMENT, "need B >= 1 and 1 <= N <= ld");
  int rc = check_filter_scalars(op, m, a, b, a0);
  if (rc) return rc;
  API_TRY
  const size_t elt = op->precision == 64 ? 8 : 4;
  // Pipeline width: the copies of chunk i+1 / i-1 overlap the filter of chunk i on two streams.  A job of fewer than
  // four chunks is cut into (up to) four narrower ones (multiples of 32 columns, at least 64) so that a single-chunk
  // job overlaps its transfers too; columns are independent, so the result does not change.
  int64_t Bc = std::min(B, N);
  if (N < 4 * Bc) {
    const int64_t quarter = ((N + 3) / 4 + 31) / 32 * 32;
    Bc = std::min(Bc, std::max<int64_t>(64, quarter));
  }
  const int64_t ldd = (Bc + 7) / 8 * 8;
  const WsLayout w = ws_layout(op, Bc);
  cudaError_t ce = cudaSuccess;
  rc = CHFSI_OK;
  const int nbuf = (N > Bc) ? 2 : 1;
  const size_t stage_need = (size_t)op->n_dofs * ldd * elt;
  for (int i = 0; i < nbuf && ce == cudaSuccess; ++i) {
    if (op->host_stage_bytes[i] < stage_need) {
      cudaFree(op->host_stage[i]); op->host_stage[i] = nullptr; op->host_stage_bytes[i] = 0;
      ce = cudaMalloc(&op->host_stage[i], stage_need);
      if (ce == cudaSuccess) op->host_stage_bytes[i] = stage_need;
    }
    if (ce == cudaSuccess && !op->host_st[i]) ce = cudaStreamCreateWithFlags(&op->host_st[i], cudaStreamNonBlocking);
    if (ce == cudaSuccess && !op->host_done[i]) ce = cudaEventCreateWithFlags(&op->host_done[i], cudaEventDisableTiming);
    // earlier asynchronous work on this handle (any stream) comes first
    if (ce == cudaSuccess && op->order_valid) ce = cudaStreamWaitEvent(op->host_st[i], op->order_ev, 0);
  }
  if (ce == cudaSuccess && op->host_ws_bytes < w.total) {
    cudaFree(op->host_ws); op->host_ws = nullptr; op->host_ws_bytes = 0;
    ce = cudaMalloc(&op->host_ws, w.total);
    if (ce == cudaSuccess) op->host_ws_bytes = w.total;
  }
  if (ce != cudaSuccess) rc = cuda_fail(op, ce, "chebyshev_filter_host allocation");
  void** stage = op->host_stage;
  void* ws = op->host_ws;
  cudaStream_t* st = op->host_st;
  cudaEvent_t* done = op->host_done;
  // The filters themselves are serialised through the single workspace by the `done` events.
  int64_t chunk = 0;
  for (int64_t j0 = 0; j0 < N && rc == CHFSI_OK; j0 += Bc, ++chunk) {
    const int s = (int)(chunk % nbuf);
    const int64_t bw = std::min(Bc, N - j0);
    char* hp = reinterpret_cast<char*>(X_host) + (size_t)j0 * elt;
    ce = cudaMemcpy2DAsync(stage[s], (size_t)ldd * elt, hp, (size_t)ldx * elt, (size_t)bw * elt, (size_t)op->n_dofs,
                           cudaMemcpyHostToDevice, st[s]);
    if (ce == cudaSuccess && chunk > 0) ce = cudaStreamWaitEvent(st[s], done[(chunk - 1) % nbuf], 0);
    if (ce != cudaSuccess) { rc = cuda_fail(op, ce, "chebyshev_filter_host H2D"); break; }
    rc = filter_block(op, stage[s], ldd, bw, m, a, b, a0, ws, st[s]);
    if (rc) break;
    ce = cudaEventRecord(done[s], st[s]);
    if (ce == cudaSuccess)
      ce = cudaMemcpy2DAsync(hp, (size_t)ldx * elt, stage[s], (size_t)ldd * elt, (size_t)bw * elt, (size_t)op->n_dofs,
                             cudaMemcpyDeviceToHost, st[s]);
    if (ce != cudaSuccess) { rc = cuda_fail(op, ce, "chebyshev_filter_host D2H"); break; }
  }
  for (int i = 0; i < nbuf; ++i)
    if (st[i]) {
      ce = cudaStreamSynchronize(st[i]);
      if (ce != cudaSuccess && rc == CHFSI_OK) rc = cuda_fail(op, ce, "chebyshev_filter_host sync");
    }
  return rc;
  API_CATCH(op)
}

namespace {
int check_rr_args(chfsi_op* op, const void* Y, int64_t ldy, int64_t N, const void* out) {
  if (!op) return CHFSI_ERR_BAD_ARGUMENT;
  if (!Y || !out) return fail(op, CHFSI_ERR_BAD_ARGUMENT, "NULL block / output matrix");
  if (N < 1 || ldy < N || N > (1 << 20)) return fail(op, CHFSI_ERR_BAD_ARGUMENT, "need 1 <= N <= ld");
  if (op->precision != 64) return fail(op, CHFSI_ERR_UNSUPPORTED, "Rayleigh-Ritz projection: FP64 operators only");
  if (N % 2 != 0 || ldy % 2 != 0 || (uintptr_t)Y % 16 != 0 || (uintptr_t)out % 16 != 0)
    return fail(op, CHFSI_ERR_UNSUPPORTED, "Rayleigh-Ritz projection: N and ld must be even, pointers 16-byte aligned");
  return CHFSI_OK;
}
}  // namespace

int chfsi_overlap_matrix(chfsi_op* op, const void* Y_dev, int64_t ldy, int64_t N, double* S_dev, void* cuda_stream) {
  if (op && op->kpoint) return fail(op, CHFSI_ERR_UNSUPPORTED, "real-block entry point called on a k-point handle");
  int rc = check_rr_args(op, Y_dev, ldy, N, S_dev);
  if (rc) return rc;
  API_TRY
  const double* Y = reinterpret_cast<const double*>(Y_dev);
  cudaStream_t st = reinterpret_cast<cudaStream_t>(cuda_stream);
  cudaError_t ce = order_enter(op, st);
  // S is Hermitian: lower triangle computed, upper mirrored
  if (ce == cudaSuccess) ce = launch_xty(op, Y, ldy, Y, ldy, op->n_dofs, (int)N, (int)N, S_dev, N, st, 1);
  if (ce == cudaSuccess) ce = launch_mirror_lower(op, S_dev, (int)N, N, st);
  if (ce == cudaSuccess) ce = order_leave(op, st);
  return ce == cudaSuccess ? CHFSI_OK : cuda_fail(op, ce, "overlap_matrix");
  API_CATCH(op)
}

int chfsi_overlap_matrix_noalloc(chfsi_op* op, const void* Y_dev, int64_t ldy, int64_t N, double* S_dev, void* cuda_stream) {
  if (op && op->kpoint) return fail(op, CHFSI_ERR_UNSUPPORTED, "real-block entry point called on a k-point handle");
  int rc = check_rr_args(op, Y_dev, ldy, N, S_dev);
  if (rc) return rc;
  if (N > CHFSI_NOALLOC_MAX_N)
    return fail(op, CHFSI_ERR_BAD_ARGUMENT,
                "overlap_matrix_noalloc: N = " + std::to_string(N) + " exceeds CHFSI_NOALLOC_MAX_N = " +
                    std::to_string(CHFSI_NOALLOC_MAX_N) + " (static scratch of 16 MiB); use chfsi_overlap_matrix");
  API_TRY
  // no order_enter / order_leave (the latter may create an event): the caller orders calls that share the static array
  cudaError_t ce = launch_xty_static(op, reinterpret_cast<const double*>(Y_dev), ldy, op->n_dofs, (int)N, S_dev, N,
                                     reinterpret_cast<cudaStream_t>(cuda_stream));
  if (ce == cudaErrorInvalidDevice)
    return fail(op, CHFSI_ERR_CUDA, "overlap_matrix_noalloc: the current device is not the one this handle was created on");
  return ce == cudaSuccess ? CHFSI_OK : cuda_fail(op, ce, "overlap_matrix_noalloc");
  API_CATCH(op)
}

int chfsi_projected_hamiltonian(chfsi_op* op, const void* Y_dev, int64_t ldy, int64_t N, int64_t B, double* H_dev,
                                void* workspace_dev, void* cuda_stream) {
  if (op && op->kpoint) return fail(op, CHFSI_ERR_UNSUPPORTED, "real-block entry point called on a k-point handle");
  int rc = check_rr_args(op, Y_dev, ldy, N, H_dev);
  if (rc) return rc;
  if (B < 2 || B % 2 != 0) return fail(op, CHFSI_ERR_BAD_ARGUMENT, "chunk width B must be even and >= 2");
  if (!workspace_dev || (uintptr_t)workspace_dev % 16 != 0) return fail(op, CHFSI_ERR_BAD_ARGUMENT, "bad workspace");
  API_TRY
  cudaStream_t st = reinterpret_cast<cudaStream_t>(cuda_stream);
  const double* Y = reinterpret_cast<const double*>(Y_dev);
  const int64_t Bc = std::min(B, N);
  const WsLayout w = ws_layout(op, Bc);
  char* base = reinterpret_cast<char*>(workspace_dev);
  double* W = reinterpret_cast<double*>(base + w.block_off);
  {
    cudaError_t ce0 = order_enter(op, st);
    if (ce0 != cudaSuccess) return cuda_fail(op, ce0, "projected_hamiltonian");
  }
  for (int64_t j0 = 0; j0 < N; j0 += Bc) {
    const int64_t bw = std::min(Bc, N - j0);
    ApplyArgs g;                                        // W <- H~ Y[:, j0 : j0 + bw]
    g.X = Y + j0; g.ldx = ldy; g.T = W; g.ldt = w.ldw; g.B = bw;
    g.alpha = 1.0; g.beta = 0.0; g.cshift = 0.0;
    g.P = base + w.p_off; g.Pc = base + w.pc_off;
    g.sync = reinterpret_cast<unsigned long long*>(base + w.sync_off); g.epoch = 1;
    cudaError_t ce = cudaMemsetAsync(g.sync, 0, w.sync_bytes, st);
    if (ce == cudaSuccess) { op->launches++; ce = launch_apply(op, g, st); }
    // H^[j0 :, j0 : j0 + bw] = Y[:, j0 :]^T W: the rows from the chunk's diagonal block down (H^ is Hermitian)
    if (ce == cudaSuccess)
      ce = launch_xty(op, Y + j0, ldy, W, w.ldw, op->n_dofs, (int)(N - j0), (int)bw, H_dev + j0 * N + j0, N, st, 1);
    if (ce != cudaSuccess) return cuda_fail(op, ce, "projected_hamiltonian");
  }
  {
    cudaError_t ce1 = launch_mirror_lower(op, H_dev, (int)N, N, st);
    if (ce1 == cudaSuccess) ce1 = order_leave(op, st);
    if (ce1 != cudaSuccess) return cuda_fail(op, ce1, "projected_hamiltonian");
  }
  return CHFSI_OK;
  API_CATCH(op)
}

int chfsi_subspace_transform(chfsi_op* op, const void* Y_dev, int64_t ldy, int64_t N, const double* Z_dev, int64_t ldz,
                             int64_t N2, void* Out_dev, int64_t ldo, void* cuda_stream) {
  if (op && op->kpoint) return fail(op, CHFSI_ERR_UNSUPPORTED, "real-block entry point called on a k-point handle");
  int rc = check_rr_args(op, Y_dev, ldy, N, Out_dev);
  if (rc) return rc;
  if (!Z_dev) return fail(op, CHFSI_ERR_BAD_ARGUMENT, "NULL transformation matrix");
  if (N2 < 1 || ldz < N2 || ldo < N2 || N2 > (1 << 20)) return fail(op, CHFSI_ERR_BAD_ARGUMENT, "need 1 <= N2 <= ldz, ldo");
  if (N2 % 2 != 0 || ldz % 2 != 0 || ldo % 2 != 0 || (uintptr_t)Z_dev % 16 != 0)
    return fail(op, CHFSI_ERR_UNSUPPORTED, "subspace_transform: N2, ldz, ldo must be even, pointers 16-byte aligned");
  const char* y0 = reinterpret_cast<const char*>(Y_dev);
  const char* o0 = reinterpret_cast<const char*>(Out_dev);
  const size_t ybytes = (size_t)op->n_dofs * ldy * 8, obytes = (size_t)op->n_dofs * ldo * 8;
  if (y0 < o0 + obytes && o0 < y0 + ybytes) return fail(op, CHFSI_ERR_BAD_ARGUMENT, "Y and Out must not overlap");
  API_TRY
  cudaStream_t st = reinterpret_cast<cudaStream_t>(cuda_stream);
  cudaError_t ce = order_enter(op, st);
  if (ce == cudaSuccess)
    ce = launch_xz(op, reinterpret_cast<const double*>(Y_dev), ldy, Z_dev, ldz, op->n_dofs, (int)N, (int)N2,
                   reinterpret_cast<double*>(Out_dev), ldo, st);
  if (ce == cudaSuccess) ce = order_leave(op, st);
  return ce == cudaSuccess ? CHFSI_OK : cuda_fail(op, ce, "subspace_transform");
  API_CATCH(op)
}

namespace {
// library-owned FP32 buffer `which` of at least `bytes` bytes (grown on demand; the stream is synchronised before a
// buffer that may still be in use is released)
cudaError_t rr32_reserve(chfsi_op* op, int which, size_t bytes, cudaStream_t st) {
  if (op->rr32_bytes[which] >= bytes) return cudaSuccess;
  cudaError_t e = cudaStreamSynchronize(st);
  if (e != cudaSuccess) return e;
  cudaFree(op->rr32[which]);
  op->rr32[which] = nullptr; op->rr32_bytes[which] = 0;
  if ((e = cudaMalloc(&op->rr32[which], bytes)) != cudaSuccess) return e;
  op->rr32_bytes[which] = bytes;
  return cudaSuccess;
}
}  // namespace

int chfsi_cholesky_inverse(chfsi_op* op, const double* S_dev, int64_t N, double* L_dev, double* Linv_dev, int* info_dev,
                           void* cuda_stream) {
  if (!op) return CHFSI_ERR_BAD_ARGUMENT;
  if (!S_dev || !L_dev || !Linv_dev || !info_dev) return fail(op, CHFSI_ERR_BAD_ARGUMENT, "NULL matrix / status pointer");
  if (N < 1 || N > 16384) return fail(op, CHFSI_ERR_BAD_ARGUMENT, "need 1 <= N <= 16384");
  if (S_dev == L_dev || S_dev == Linv_dev || L_dev == Linv_dev) return fail(op, CHFSI_ERR_BAD_ARGUMENT, "S, L and L^-1 must be distinct arrays");
  API_TRY
  cudaStream_t st = reinterpret_cast<cudaStream_t>(cuda_stream);
  cudaError_t ce = order_enter(op, st);
  if (ce == cudaSuccess) ce = launch_cholesky_inverse(op, S_dev, (int)N, L_dev, Linv_dev, info_dev, st);
  if (ce == cudaSuccess) ce = order_leave(op, st);
  return ce == cudaSuccess ? CHFSI_OK : cuda_fail(op, ce, "cholesky_inverse");
  API_CATCH(op)
}

int chfsi_overlap_matrix_mixed(chfsi_op* op, const void* Y_dev, int64_t ldy, int64_t N, int64_t block, double* S_dev,
                               void* cuda_stream) {
  if (op && op->kpoint) return fail(op, CHFSI_ERR_UNSUPPORTED, "real-block entry point called on a k-point handle");
  int rc = check_rr_args(op, Y_dev, ldy, N, S_dev);
  if (rc) return rc;
  if (block < 2 || block % 2 != 0) return fail(op, CHFSI_ERR_BAD_ARGUMENT, "block width must be even and >= 2");
  API_TRY
  cudaStream_t st = reinterpret_cast<cudaStream_t>(cuda_stream);
  const double* Y = reinterpret_cast<const double*>(Y_dev);
  const int64_t ld32 = (N + 3) / 4 * 4;
  cudaError_t ce = order_enter(op, st);
  if (ce == cudaSuccess) ce = rr32_reserve(op, 0, (size_t)op->n_dofs * ld32 * sizeof(float), st);
  float* Y32 = reinterpret_cast<float*>(op->rr32[0]);
  if (ce == cudaSuccess) ce = launch_to_f32(op, Y, ldy, Y32, ld32, op->n_dofs, (int)N, 0, nullptr, st);
  // FP32 blocks first (tiles inside a diagonal block are skipped), then the FP64 diagonal blocks on top
  // (lower triangle only, mirrored at the end: PAPER.md:558)
  if (ce == cudaSuccess) ce = launch_xty_tf32(op, Y32, ld32, Y32, ld32, op->n_dofs, (int)N, (int)N, (int)block, 0, 0, S_dev, N, st, 1);
  for (int64_t j0 = 0; j0 < N && ce == cudaSuccess; j0 += block) {
    const int bw = (int)std::min(block, N - j0);
    ce = launch_xty(op, Y + j0, ldy, Y + j0, ldy, op->n_dofs, bw, bw, S_dev + j0 * N + j0, N, st, 1);
  }
  if (ce == cudaSuccess) ce = launch_mirror_lower(op, S_dev, (int)N, N, st);
  if (ce == cudaSuccess) ce = order_leave(op, st);
  return ce == cudaSuccess ? CHFSI_OK : cuda_fail(op, ce, "overlap_matrix_mixed");
  API_CATCH(op)
}

int chfsi_projected_hamiltonian_mixed(chfsi_op* op, const void* Y_dev, int64_t ldy, int64_t N, int64_t B, int64_t n_oc,
                                      double* H_dev, void* workspace_dev, void* cuda_stream) {
  if (op && op->kpoint) return fail(op, CHFSI_ERR_UNSUPPORTED, "real-block entry point called on a k-point handle");
  int rc = check_rr_args(op, Y_dev, ldy, N, H_dev);
  if (rc) return rc;
  if (B < 2 || B % 2 != 0) return fail(op, CHFSI_ERR_BAD_ARGUMENT, "chunk width B must be even and >= 2");
  if (n_oc < 0 || n_oc > N || n_oc % 2 != 0) return fail(op, CHFSI_ERR_BAD_ARGUMENT, "need 0 <= n_oc <= N, n_oc even");
  if (!workspace_dev || (uintptr_t)workspace_dev % 16 != 0) return fail(op, CHFSI_ERR_BAD_ARGUMENT, "bad workspace");
  API_TRY
  cudaStream_t st = reinterpret_cast<cudaStream_t>(cuda_stream);
  const double* Y = reinterpret_cast<const double*>(Y_dev);
  const int64_t Bc = std::min(B, N);
  const WsLayout w = ws_layout(op, Bc);
  char* base = reinterpret_cast<char*>(workspace_dev);
  double* W = reinterpret_cast<double*>(base + w.block_off);
  const int64_t ld32 = (N + 3) / 4 * 4, ldw32 = (Bc + 3) / 4 * 4;
  cudaError_t ce = order_enter(op, st);
  if (ce == cudaSuccess) ce = rr32_reserve(op, 0, (size_t)op->n_dofs * ld32 * sizeof(float), st);
  if (ce == cudaSuccess) ce = rr32_reserve(op, 1, (size_t)op->n_dofs * ldw32 * sizeof(float), st);
  float* Y32 = reinterpret_cast<float*>(op->rr32[0]);
  float* W32 = reinterpret_cast<float*>(op->rr32[1]);
  if (ce == cudaSuccess) ce = launch_to_f32(op, Y, ldy, Y32, ld32, op->n_dofs, (int)N, 0, nullptr, st);
  for (int64_t j0 = 0; j0 < N && ce == cudaSuccess; j0 += Bc) {
    const int64_t bw = std::min(Bc, N - j0);
    ApplyArgs g;                                        // W <- H~ Y[:, j0 : j0 + bw]   (FP64)
    g.X = Y + j0; g.ldx = ldy; g.T = W; g.ldt = w.ldw; g.B = bw;
    g.alpha = 1.0; g.beta = 0.0; g.cshift = 0.0;
    g.P = base + w.p_off; g.Pc = base + w.pc_off;
    g.sync = reinterpret_cast<unsigned long long*>(base + w.sync_off); g.epoch = 1;
    ce = cudaMemsetAsync(g.sync, 0, w.sync_bytes, st);
    if (ce == cudaSuccess) { op->launches++; ce = launch_apply(op, g, st); }
    // Eq. 39: all rows of these columns as FP32 products ...
    if (ce == cudaSuccess) ce = launch_to_f32(op, W, w.ldw, W32, ldw32, op->n_dofs, (int)bw, 0, nullptr, st);
    // (rows from the chunk's diagonal block down: H^ is Hermitian; the first row is rounded down to a multiple
    // of 4 for the 16-byte alignment of the FP32 operand, so up to two rows above the diagonal block are computed as well)
    const int64_t r0 = j0 / 4 * 4;
    if (ce == cudaSuccess)
      ce = launch_xty_tf32(op, Y32 + r0, ld32, W32, ldw32, op->n_dofs, (int)(N - r0), (int)bw, 0, 0, 0, H_dev + r0 * N + j0, N, st, 1);
    // ... and the fr-fr part (rows and columns >= n_oc) in FP64 on top
    const int64_t c0 = std::max(j0, n_oc);
    if (ce == cudaSuccess && c0 < j0 + bw && n_oc < N)
      ce = launch_xty(op, Y + c0, ldy, W + (c0 - j0), w.ldw, op->n_dofs, (int)(N - c0), (int)(j0 + bw - c0),
                      H_dev + c0 * N + c0, N, st, 1);
  }
  if (ce == cudaSuccess) ce = launch_mirror_lower(op, H_dev, (int)N, N, st);
  if (ce == cudaSuccess) ce = order_leave(op, st);
  return ce == cudaSuccess ? CHFSI_OK : cuda_fail(op, ce, "projected_hamiltonian_mixed");
  API_CATCH(op)
}

int chfsi_subspace_transform_mixed(chfsi_op* op, const void* Y_dev, int64_t ldy, int64_t N, const double* Z_dev, int64_t ldz,
                                   void* Out_dev, int64_t ldo, void* cuda_stream) {
  if (op && op->kpoint) return fail(op, CHFSI_ERR_UNSUPPORTED, "real-block entry point called on a k-point handle");
  int rc = check_rr_args(op, Y_dev, ldy, N, Out_dev);
  if (rc) return rc;
  if (!Z_dev) return fail(op, CHFSI_ERR_BAD_ARGUMENT, "NULL transformation matrix");
  if (ldz < N || ldo < N) return fail(op, CHFSI_ERR_BAD_ARGUMENT, "need N <= ldz, ldo");
  if (ldz % 2 != 0 || ldo % 2 != 0 || (uintptr_t)Z_dev % 16 != 0)
    return fail(op, CHFSI_ERR_UNSUPPORTED, "subspace_transform_mixed: ldz, ldo must be even, pointers 16-byte aligned");
  const char* y0 = reinterpret_cast<const char*>(Y_dev);
  const char* o0 = reinterpret_cast<const char*>(Out_dev);
  const size_t ybytes = (size_t)op->n_dofs * ldy * 8, obytes = (size_t)op->n_dofs * ldo * 8;
  if (y0 < o0 + obytes && o0 < y0 + ybytes) return fail(op, CHFSI_ERR_BAD_ARGUMENT, "Y and Out must not overlap");
  API_TRY
  cudaStream_t st = reinterpret_cast<cudaStream_t>(cuda_stream);
  const double* Y = reinterpret_cast<const double*>(Y_dev);
  const int64_t ld32 = (N + 3) / 4 * 4;
  cudaError_t ce = order_enter(op, st);
  if (ce == cudaSuccess) ce = rr32_reserve(op, 0, (size_t)op->n_dofs * ld32 * sizeof(float), st);
  // FP32 copy of Z without its diagonal, followed by the FP64 diagonal, in the second buffer
  const size_t z32_bytes = align_up((size_t)N * ld32 * sizeof(float), 256);
  if (ce == cudaSuccess) ce = rr32_reserve(op, 1, z32_bytes + (size_t)N * sizeof(double), st);
  float* Y32 = reinterpret_cast<float*>(op->rr32[0]);
  float* Z32 = reinterpret_cast<float*>(op->rr32[1]);
  double* zd = reinterpret_cast<double*>(reinterpret_cast<char*>(op->rr32[1]) + z32_bytes);
  if (ce == cudaSuccess) ce = launch_to_f32(op, Y, ldy, Y32, ld32, op->n_dofs, (int)N, 0, nullptr, st);
  if (ce == cudaSuccess) ce = launch_to_f32(op, Z_dev, ldz, Z32, ld32, N, (int)N, 1, zd, st);
  if (ce == cudaSuccess)
    ce = launch_xz_tf32(op, Y32, ld32, Z32, ld32, Y, ldy, zd, op->n_dofs, (int)N, (int)N, reinterpret_cast<double*>(Out_dev), ldo, st);
  if (ce == cudaSuccess) ce = order_leave(op, st);
  return ce == cudaSuccess ? CHFSI_OK : cuda_fail(op, ce, "subspace_transform_mixed");
  API_CATCH(op)
}

int64_t chfsi_launch_count(const chfsi_op* op) { return op ? op->launches : -1; }

int chfsi_set_kernel_variant(chfsi_op* op, int variant) {
  if (!op) return CHFSI_ERR_BAD_ARGUMENT;
  if (variant < 0 || variant > 6) return fail(op, CHFSI_ERR_BAD_ARGUMENT, "variant must be 0 .. 6");
  op->variant = variant;
  return CHFSI_OK;
}

int chfsi_set_rr_variant(chfsi_op* op, int variant) {
  if (!op) return CHFSI_ERR_BAD_ARGUMENT;
  if (variant < 0 || variant > 2) return fail(op, CHFSI_ERR_BAD_ARGUMENT, "rr variant must be 0 .. 2");
  op->rr_variant = variant;
  return CHFSI_OK;
}

int chfsi_set_profiling(chfsi_op* op, int enabled) {
  if (!op) return CHFSI_ERR_BAD_ARGUMENT;
  op->profiling = enabled != 0;
  op->prof_used = 0; op->prof_main_launches = 0; op->prof_proj_launches = 0;
  return CHFSI_OK;
}

int chfsi_get_profile(chfsi_op* op, chfsi_profile* prof) {
  if (!op || !prof) return CHFSI_ERR_BAD_ARGUMENT;
  API_TRY
  std::memset(prof, 0, sizeof(*prof));
  for (size_t i = 0; i + 3 <= op->prof_used; i += 3) {
    cudaError_t ce = cudaEventSynchronize(op->prof_events[i + 2]);
    if (ce != cudaSuccess) return cuda_fail(op, ce, "get_profile");
    float ms_p = 0.f, ms_m = 0.f;
    cudaEventElapsedTime(&ms_p, op->prof_events[i], op->prof_events[i + 1]);
    cudaEventElapsedTime(&ms_m, op->prof_events[i + 1], op->prof_events[i + 2]);
    prof->projector_ms += ms_p; prof->contraction_ms += ms_m; prof->applies++;
  }
  prof->contraction_launches = op->prof_main_launches; prof->projector_launches = op->prof_proj_launches;
  op->prof_used = 0; op->prof_main_launches = 0; op->prof_proj_launches = 0;
  return CHFSI_OK;
  API_CATCH(op)
}

const char* chfsi_last_error(const chfsi_op* op) { return op ? op->err.c_str() : g_create_error.c_str(); }

}  // extern "C"
