// Internal declarations shared by the translation units of libchfsi (not part of the ABI).
//
// Device data layout:
//   mat   [cell c]  : [n_parts] blocks of K_c rows x LDA columns (block = mw consecutive output nodes; one block up to
//                     p = 6); per block: K_c rows x LDA columns, element type T (double | float), row k = CONTRACTION index,
//                     column m = OUTPUT node.  Rows 0..M_cell-1 hold the Loewdin-scaled cell Hamiltonian
//                     s_k H^e_km s_m (symmetric, "H~^{loc,c_i}"); rows M_cell..M_cell+N_psp^c-1
//                     hold s_m C^c_{m,j} for the projectors j touching the cell; remaining
//                     rows/columns are zero padding.  K_c is a multiple of 8, LDA = round8(M_cell) + 4 so that
//                     FP64 mma fragments read shared memory without bank conflicts (LDA mod 16 in {4, 12}).
//   gidx  [cell c]  : K_c int32.  k < M_cell: global dof of local node k, bit 31 set when this (cell, node) is
//                     the FIRST contribution to that dof in colour order (it then carries the recurrence
//                     terms); k >= M_cell: row of the projector-coefficient block P (padding rows point at
//                     the all-zero row n_proj).
//   X, Y  blocks    : [n_dofs][ld], vector index fastest.
//   P               : [n_proj + 1][B]   (Alg. 4 steps 3-4: assembled and D-scaled projector coefficients)
//   Pc              : [nnz_cell_proj][B] (Alg. 4 step 2: per-cell partial coefficients C^cT X^c)
#pragma once
#include <cstdint>
#include <string>
#include <vector>

#include <cuda_runtime.h>

#include "../../include/chfsi.h"

namespace chfsi {

constexpr uint32_t kFirstBit = 0x80000000u;
constexpr int kMaxPartMTiles = 44;       // 8-row output tiles per part (4 warp rows x 11)
// element offset of (contraction row k, output column m) inside the matrix of a cell with K_c = kc rows
__host__ __device__ inline int64_t mat_elem(int k, int m, int mw, int lda, int kc) {
  return (int64_t)(m / mw) * kc * lda + (int64_t)k * lda + (m % mw);
}
constexpr int kProjGroup = 8;            // projectors per group (slots of a coefficient row)
constexpr int kProjSegRows = 128;        // dof rows per CTA of the projector-coefficient kernel

// ---- host-side tables and mesh analysis (host_setup.cpp) -------------------------------------------------
struct Tables1D {
  int p = 0, n1 = 0, nq1 = 0;
  std::vector<double> gll_x, gll_w;   // [n1]
  std::vector<double> gq_x, gq_w;     // [nq1]
  std::vector<double> phi, dphi;      // [nq1][n1]  Lagrange (GLL) basis and derivative at the Gauss points
};
void build_tables(int p, Tables1D* t);

struct HostPlan {
  // colouring
  int n_colors = 0;
  std::vector<int32_t> color_cells;      // cells sorted by colour
  std::vector<int32_t> color_ptr;        // [n_colors+1]
  // assembly dependencies by position in colour order (CSR): earlier positions that share a dof
  std::vector<int32_t> dep_ptr;          // [n_cells+1]
  std::vector<int32_t> dep_pos;
  // cell-centric projector lists
  std::vector<int64_t> cell_proj_ptr;    // [n_cells+1]
  std::vector<int32_t> cell_proj_idx;    // [nnz] projector id
  std::vector<int64_t> cell_proj_src;    // [nnz] index k into the caller's (projector,cell) CSR (chi_q row)
  // per-cell layout
  std::vector<int32_t> ktot;             // [n_cells]
  std::vector<int64_t> mat_off;          // [n_cells+1] element offsets into mat
  std::vector<int64_t> idx_off;          // [n_cells+1] offsets into gidx
  std::vector<int32_t> gidx;
  // projector-centric reduction lists (Alg. 4 step 3)
  std::vector<int64_t> proj_ptr;         // [n_proj+1]
  std::vector<int64_t> proj_pcrow;       // [nnz] row of Pc
  std::vector<int32_t> pc_cells;         // cells that have projectors
  // dof-centric projector lists: projectors with the same support (one atom's) form a group of <= 8; the rows of a
  // group are the dofs of its support cells; the assembly over cells of Alg. 4 step 3 is applied to
  // C ONCE at setup (coefficients s_g sum_c C^c[l(g)][j]), so that per apply every dof row of X is read once per
  // group instead of once per (cell, group).  Segments of <= kProjSegRows rows are the CTAs of k_proj_rows.
  int n_groups = 0;
  std::vector<int32_t> grp_row_ptr;      // [n_groups+1]
  std::vector<int32_t> grow_dof;         // [n_rows] global dof, ascending inside a group
  std::vector<int32_t> grp_proj;         // [n_groups][8] projector ids, -1 = unused slot
  std::vector<int32_t> seg_ptr;          // [n_seg+1] row ranges; a segment never straddles two groups
  std::vector<int32_t> grp_seg_ptr;      // [n_groups+1]
  std::vector<int32_t> proj_grp, proj_slot;   // [n_proj]
  std::vector<double> mass;              // [n_dofs] diagonal GLL mass
};
// Returns "" on success, else an error message (bad mesh).
std::string analyse_mesh(const chfsi_mesh& mesh, const chfsi_nonlocal* nl, const Tables1D& tab, int lda, int n_parts,
                         HostPlan* plan);
// Diagonal GLL mass of a mesh on the host; returns an error text or "".
std::string mesh_mass(const chfsi_mesh& mesh, const Tables1D& tab, std::vector<double>* mass);

// ---- device operator ----------------------------------------------------------------------------------------
struct Op {
  int p = 0, n1 = 0, nq1 = 0, m_cell = 0, n_q = 0, mpad = 0, lda = 0;
  // output columns of a cell matrix are stored in n_parts blocks of mw columns: mat[c] = [part][K_c][lda]
  // (one block, mw = mpad, up to p = 6; two blocks of 256 at p = 7, three of 248 at p = 8): a tile of the persistent
  // kernel is (cell, part, column tile), so the accumulators of 8 warps always fit the register file.
  int n_parts = 1, mw = 0;
  int precision = 64, assembly = 0, variant = 0;
  int rr_variant = 0;                    // FP32 blocks of the mixed Rayleigh-Ritz products: 0 / 1 tcgen05 (rr_umma.cu), 2 mma.sync
  int64_t n_cells = 0, n_dofs = 0, n_proj = 0, nnz_cp = 0, n_pc_cells = 0;
  int n_colors = 0;
  std::vector<int32_t> color_ptr;        // host copy
  int max_ktot = 0;
  int64_t mat_elems = 0;
  // device arrays
  void* mat = nullptr;                   // T
  int64_t* mat_off = nullptr;
  int64_t* idx_off = nullptr;
  int32_t* ktot = nullptr;
  int32_t* gidx = nullptr;
  int32_t* color_cells = nullptr;
  int32_t* dep_ptr = nullptr;            // [n_cells+1] by position in colour order
  int32_t* dep_pos = nullptr;
  int n_sm = 0;
  int32_t* all_cells = nullptr;          // 0..n_cells-1 (atomic mode launches every cell at once)
  int32_t* pc_cells = nullptr;
  int64_t* cell_proj_ptr = nullptr;      // [n_cells+1]  (row offsets into Pc)
  int64_t* proj_ptr = nullptr;
  int64_t* proj_pcrow = nullptr;
  // dof-centric projector data (HostPlan): segments, rows, assembled coefficients [n_prow][8] (element type T)
  int64_t n_pseg = 0, n_prow = 0;
  int32_t* seg_ptr = nullptr;
  int32_t* grow_dof = nullptr;
  void* pcoef = nullptr;
  int32_t* grp_seg_ptr = nullptr;
  int32_t* proj_grp = nullptr;
  int32_t* proj_slot = nullptr;
  double* D = nullptr;
  double* mass = nullptr;
  // Spectral shift folded into the cell matrices: diag0 [n_cells][m_cell] keeps the unshifted diagonal entries
  // mat[c][k][k]; while a filter runs, the diagonal entry of the (cell, node) that makes the FIRST contribution
  // to its dof holds diag0 - cur_shift, so that the contraction itself yields (H~ - c I) X  (Eq. 37's
  // "c1 H~ + c2") and the recurrence epilogue never re-reads X.
  double* diag0 = nullptr;
  double cur_shift = 0.0;
  // sum-factorised variant (apply_sf.cuh; FE degree <= 6): quadrature-point fields W0 = w detJ V_eff and
  // G = 1/2 w detJ J^-1 J^-T in the kernel's lane order [n_cells][nq1][7][32][2], M^-1/2 per (cell, node)
  // [n_cells][mpad], and the projector columns s_l C^c_{l,j} as compact FP64 rows [nnz_cp][m_cell]
  bool sf_ok = false;
  // chfsi_update_potential on an operator whose default kernel is sum-factorised only refreshes the quadrature-point fields
  // (veff_dev keeps the samples on the device); the dense cell matrices are rebuilt from veff_dev the first time a dense
  // kernel variant is asked for afterwards
  double* veff_dev = nullptr;            // [n_cells][n_q], set by the first chfsi_update_potential
  bool dense_stale = false;
  // k-point variant (chfsi_create_k): vector blocks are complex (FP64 pairs re, im = two adjacent real columns), the
  // fields carry w detJ J^-1 k, the projector coefficients are complex (pcoef = real parts, pcoef_im = imaginary parts) and
  // the back-projection C (D P) runs as its own dof-centric kernel (k_proj_back), one launch per colour of the projector groups
  bool kpoint = false;
  double kvec[3] = {0.0, 0.0, 0.0};
  void* pcoef_im = nullptr;              // [n_prow][8]
  int32_t* seg_slot_proj = nullptr;      // [n_pseg][8] projector (row of P) of slot i of the segment's group, -1 if empty
  int32_t* back_segs = nullptr;          // segments ordered by the colour of their group
  std::vector<int32_t> back_color_ptr;   // [n_back_colors + 1] into back_segs
  double* sf_coef = nullptr;
  double* sf_sloc = nullptr;
  double* crows = nullptr;
  // kept from create for chfsi_update_potential: cell vertices and the 1-D tables of the setup kernels
  double* setup_verts = nullptr;         // [n_cells][24]
  double* setup_pp = nullptr;            // [4][nq1][n1*n1]
  double* setup_phi = nullptr;           // [nq1][n1]
  double* setup_gx = nullptr;            // [nq1]
  double* setup_gw = nullptr;            // [nq1]
  // split-row partial tiles of the Rayleigh-Ritz projection products (rr_kernels.cu); grown on demand
  void* rr_scratch = nullptr;
  int* rr_flag = nullptr;             // device word: != 0 when the Z of the current Y Z product has a nonzero below its diagonal
  size_t rr_scratch_bytes = 0;
  // FP32 copies of the blocks of the mixed-precision Rayleigh-Ritz products; grown on demand
  void* rr32[2] = {nullptr, nullptr};
  size_t rr32_bytes[2] = {0, 0};
  // device staging of chfsi_chebyshev_filter_host, kept between calls (grown on demand, freed at destroy)
  void* host_stage[2] = {nullptr, nullptr};
  size_t host_stage_bytes[2] = {0, 0};
  void* host_ws = nullptr;
  size_t host_ws_bytes = 0;
  cudaStream_t host_st[2] = {nullptr, nullptr};
  cudaEvent_t host_done[2] = {nullptr, nullptr};
  // cross-stream ordering of the calls on this handle (api.cu order_enter / order_leave)
  cudaEvent_t order_ev = nullptr;
  cudaStream_t order_stream = nullptr;
  bool order_valid = false;
  int64_t launches = 0;
  // optional per-kernel timing (chfsi_set_profiling): event triples (start, after projector kernels, end)
  bool profiling = false;
  std::vector<cudaEvent_t> prof_events;
  size_t prof_used = 0;
  int64_t prof_main_launches = 0, prof_proj_launches = 0;
  std::string err;
};

// ---- setup kernels (setup_kernels.cu) ------------------------------------------------------------------------
// Fills op->mat (element type per op->precision) from the mesh geometry, V_eff and projector samples.
// All pointer arguments are HOST pointers except op's device arrays.  Returns cudaSuccess or the failing code;
// *bad_jacobian is set when some quadrature point has det J <= 0.
cudaError_t build_cell_matrices(Op* op, const HostPlan& plan, const Tables1D& tab, const chfsi_mesh& mesh,
                                const chfsi_potential& pot, const chfsi_nonlocal* nl, cudaStream_t stream,
                                bool* bad_jacobian);
// Recomputes the Hamiltonian rows (rows 0..M_cell-1) of every cell matrix for a new V_eff (HOST pointer
// [n_cells][(p+2)^3]); projector rows, layout and colouring are untouched.  Synchronises the stream.
cudaError_t rebuild_local_matrices(Op* op, const double* veff_q_host, cudaStream_t stream);
// The same from op->veff_dev, followed by capture_diagonal: brings stale dense matrices up to date (op->dense_stale).
cudaError_t refresh_dense_matrices(Op* op, cudaStream_t stream);
// Quadrature-point fields of the sum-factorised variant (op->sf_coef, allocated on first use) from V_eff at the Gauss
// points (HOST pointer) and the cell geometry; op->setup_* must exist.  Synchronises the stream.
cudaError_t build_sf_fields(Op* op, const double* veff_q_host, cudaStream_t stream);
// The same from samples already on the device; enqueues only (no synchronisation).
cudaError_t build_sf_fields_dev(Op* op, const double* veff_q_dev, cudaStream_t stream);
// Projector rows of the cell matrices from projector samples at the Gauss points (HOST pointer); see setup_kernels.cu.
cudaError_t build_cell_projectors(Op* op, const HostPlan& plan, const double* chi_host, cudaStream_t stream);

// ---- apply kernels (apply_kernels.cu) ----------------------------------------------------------------------
struct ApplyArgs {
  const void* X = nullptr;  int64_t ldx = 0;     // input block Y_{k-1}
  void* T = nullptr;        int64_t ldt = 0;     // target block: holds Y_{k-2} on entry, Y_k on exit
  int64_t B = 0;
  double alpha = 1.0, beta = 0.0, cshift = 0.0;  // Y_k = alpha (H~ X - cshift X) - beta T
  void* P = nullptr;                             // [n_proj+1][B]
  void* Pc = nullptr;                            // [n_pseg][8][B] FP64 partial coefficients of the row segments
  // single-launch deterministic assembly: ticket counter (slot 0, 64-bit) and per-(position, column tile)
  // completion flags, zeroed by the caller of launch_apply before epoch 1; epoch increases by one per launch
  unsigned long long* sync = nullptr;
  uint32_t epoch = 0;
  // accumulate: T <- T + alpha (H~ X - cshift X); beta is ignored and the target block is never read by the kernel
  // (every contribution is a red.add).  Only the warp-specialised sum-factorised kernel takes it: ask
  // apply_accumulates() first.  The filter loop then runs the recurrence in scaled blocks (api.cu filter_block).
  bool accumulate = false;
  // phase: 0 = the whole application; 1 = steps 3a-3c only (the D-scaled projector coefficients P of this operator's cells
  // are left in the workspace rows `P`); 2 = everything but steps 3a-3c (`P` is given).  Phases 1 and 2 let a caller
  // that holds only a part of the mesh sum P over the parts in between (Alg. 4 step 3).
  int phase = 0;
};
// Helpers of the cell-partitioned filter (part_kernels.cu): rows of a block to / from a packed buffer of the block's own
// type (buf_precision == op->precision) or FP32, and one degree of the three-term recurrence on whole blocks.
cudaError_t launch_pack_rows(Op* op, const void* X, int64_t ldx, int64_t B, const int32_t* rows, const int32_t* slots,
                             int64_t n_rows, void* buf, int buf_precision, bool unpack, cudaStream_t stream);
// accumulate-only exchange: pack  buf[s(i)] = T[rows[i]] - base[i] + corr X[rows[i]] (1 - owner[i])  /  unpack
// T[rows[i]] = base[i] + buf[s(i)]   (base [n_rows][B] contiguous or nullptr; part_kernels.cu)
cudaError_t launch_rows_delta(Op* op, void* T, int64_t ldt, const void* base, const void* X, int64_t ldx, const uint8_t* owner,
                              double corr, int64_t B, const int32_t* rows, const int32_t* slots, int64_t n_rows, void* buf,
                              int buf_precision, bool unpack, cudaStream_t stream);
cudaError_t launch_recurrence(Op* op, const void* HX, int64_t ldh, const void* X, int64_t ldx, void* T, int64_t ldt, int64_t B,
                              double alpha, double beta, double c, cudaStream_t stream);
// True when launch_apply would run these arguments (X, ldx, T, ldt, P, B, sync set) with accumulate = true.
bool apply_accumulates(const Op* op, const ApplyArgs& a);
// dst[g][0..B) = factor * src[g][0..B) for all dofs g (element type per op->precision; dst may equal src).
cudaError_t launch_scale_block(Op* op, void* dst, int64_t ldd, const void* src, int64_t lds, int64_t B, double factor,
                               cudaStream_t stream);
// Enqueues one fused H~ application + recurrence update.  Returns cudaGetLastError().
cudaError_t launch_apply(Op* op, const ApplyArgs& a, cudaStream_t stream);
// Builds op->pcoef: the projector rows of the cell matrices summed over the cells of each dof (once, at create,
// after build_cell_matrices; deterministic host summation in the caller's CSR order).
cudaError_t assemble_projector_rows(Op* op, const HostPlan& plan, const chfsi_mesh& mesh, cudaStream_t stream);
// k-point variant: the same assembly for the imaginary parts (the cell matrices then hold them in their projector rows)
// into op->pcoef_im, and the group / colour tables of the back-projection kernel.
cudaError_t assemble_projector_rows_imag(Op* op, const HostPlan& plan, const chfsi_mesh& mesh, cudaStream_t stream);
// Copies the diagonal of every cell matrix into op->diag0 (once, at create, after build_cell_matrices).
cudaError_t capture_diagonal(Op* op, cudaStream_t stream);
// C[N1][ldc] = A^T B over n_rows rows of two FP64 blocks [n_rows][ld] (Alg. 2 step 1); enqueued on
// the stream; may grow op->rr_scratch (then it synchronises the stream once).
// lower != 0: the result is the lower triangle (r >= c, local indices) of a Hermitian matrix: tiles strictly above the diagonal
// are not computed and entries above it are not written; launch_mirror_lower then fills C[r][c] = C[c][r], c > r.
cudaError_t launch_xty(Op* op, const double* A, int64_t lda, const double* B, int64_t ldb, int64_t n_rows, int N1, int N2,
                       double* C, int64_t ldc, cudaStream_t stream, int lower = 0);
cudaError_t launch_mirror_lower(Op* op, double* C, int N, int64_t ldc, cudaStream_t stream);
// Allocation-free S = Y^T Y (chfsi_overlap_matrix_noalloc): partial sums in a file-scope __device__ array of rr_kernels.cu
// whose device address resolve_xty_static() looks up once per device (called by init_rr_kernels with that device current).
cudaError_t resolve_xty_static();
cudaError_t launch_xty_static(Op* op, const double* Y, int64_t ldy, int64_t n_rows, int N, double* S, int64_t lds, cudaStream_t stream);
// Out[n_rows][ldo] = Y Z, Y [n_rows][ldy] with N columns, Z [N][ldz] with N2 columns (Alg. 2 step 3)
cudaError_t launch_xz(Op* op, const double* Y, int64_t ldy, const double* Z, int64_t ldz, int64_t n_rows, int N, int N2,
                      double* Out, int64_t ldo, cudaStream_t stream);
// Mixed-precision products of the Rayleigh-Ritz step (rr_kernels.cu): FP32 operands, 3xTF32
// products, FP64 totals.  launch_to_f32 rounds an FP64 block to FP32 (optionally splitting off the diagonal of a square
// matrix); launch_xty_tf32 writes C = A^T B except the tiles inside diagonal blocks of width skip_block (> 0);
// launch_xz_tf32 writes Out = Y32 Z32 + Y diag(zd).
cudaError_t init_rr_mixed_kernels();
cudaError_t launch_to_f32(Op* op, const double* src, int64_t lds, float* dst, int64_t ldd, int64_t rows, int cols, int zero_diag,
                          double* diag, cudaStream_t st);
// tcgen05 form of the same product (rr_umma.cu): partial sums of the row splits into Cpart[n_split][N1][N2]; false when the
// tensor maps cannot be encoded (the caller then runs k_xty_tf32).  init_umma_kernels: per-device kernel attributes.
cudaError_t init_umma_kernels();
void umma_xty_plan(int n_sm, int64_t n_rows, int N1, int N2, int skip_block, int row_block0, int col_block0, int lower,
                   int* n_split, int64_t* rows_per_split);          // row splits for launch_xty_umma (rows per split: a multiple of 32)
bool launch_xty_umma(const float* A, int64_t lda, const float* B, int64_t ldb, int64_t n_rows, int N1, int N2, int n_split,
                     int64_t rows_per_split, int skip_block, int row_block0, int col_block0, int lower, double* Cpart,
                     cudaStream_t stream);
bool launch_xz_umma(const float* Y32, int64_t ldy32, const float* Z32, int64_t ldz32, const double* Y, int64_t ldy, const double* zd,
                    int64_t n_rows, int N, int N2, double* Out, int64_t ldo, const int* lower_nonzero, cudaStream_t stream);
cudaError_t launch_xty_tf32(Op* op, const float* A, int64_t lda, const float* B, int64_t ldb, int64_t n_rows, int N1, int N2,
                            int skip_block, int row_block0, int col_block0, double* C, int64_t ldc, cudaStream_t st, int lower = 0);
cudaError_t launch_xz_tf32(Op* op, const float* Y32, int64_t ldy32, const float* Z32, int64_t ldz32, const double* Y, int64_t ldy,
                           const double* zd, int64_t n_rows, int N, int N2, double* Out, int64_t ldo, cudaStream_t st);
// Cholesky factor and its inverse of an N x N FP64 matrix on the device (rr_dense.cu; Alg. 2 step 2a)
cudaError_t launch_cholesky_inverse(Op* op, const double* S, int N, double* L, double* Linv, int* info_dev, cudaStream_t st);
// Opts the kernels into the shared memory they need for this operator, on the CURRENT device (at every create: the
// attribute is per device).
cudaError_t init_apply_kernels(Op* op);
cudaError_t init_rr_kernels();
// Sum-factorised variant: uploads the 1-D tables of degree tab.p to constant memory of the current device and fills
// op->sf_sloc; sets op->sf_ok when the operator qualifies (p <= 6, at most kSfMaxProj projectors per cell).
cudaError_t init_sf_variant(Op* op, const Tables1D& tab, cudaStream_t stream);

}  // namespace chfsi
