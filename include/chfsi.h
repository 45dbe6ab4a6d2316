/* chfsi.h -- C ABI of the B200-native Chebyshev-filter hot path of DFT-FE (arxiv 2203.07820).
 *
 * Citations are PAPER.md:<line> (= /root/reference/PAPER.md) plus the section / equation / algorithm.
 *
 * What the library computes
 * -------------------------
 *   H~ = M^-1/2 ( 1/2 K + V_eff + sum_a C_a D_a C_a^T ) M^-1/2           Eq. 30 terms 1-2,
 *                                                                         Eq. 33, Eq. 34
 *   apply_H :          Y = H~ X                                           Eq. 47, Alg. 4
 *   chebyshev_filter : X <- T_m((H~ - c)/e) X / T_m((a0 - c)/e),  e=(b-a)/2, c=(b+a)/2
 *                      Eq. 37 in the scaled three-term form of ref. [86]:
 *                        sigma_1 = e/(a0-c);  Y_1 = (sigma_1/e)(H~ X - c X)
 *                        sigma_k = 1/(2/sigma_1 - sigma_{k-1})
 *                        Y_k = (2 sigma_k/e)(H~ Y_{k-1} - c Y_{k-1}) - sigma_{k-1} sigma_k Y_{k-2},  k = 2..m
 *
 * on a hexahedral spectral-element mesh (GLL nodes) with the diagonal GLL mass matrix M
 * (PAPER.md:336), K and V_eff integrated with (p+2)^3 Gauss-Legendre points, cell by cell:
 * extraction -> per-cell dense product with the Loewdin-scaled cell matrix -> assembly.
 *
 * Conventions
 * -----------
 *  - Every call returns an int: CHFSI_OK (0) or a negative chfsi_status.  Nothing throws or aborts across
 *    the ABI.  chfsi_last_error() gives a human-readable message for the last failing call on a handle
 *    (or for a failed chfsi_create when passed NULL).
 *  - Vectors live in the Loewdin space x~ = M^{1/2} x^.  A block of vectors is a row-major
 *    array [n_dofs][ld] with the VECTOR INDEX FASTEST; ld >= B, so a chunk of B columns of a
 *    wider array is addressed by passing a pointer to its first column and the wide array's ld.
 *    Element type is double (precision 64) or float (precision 32).
 *  - "_dev" pointers are device pointers owned by the CALLER (PyTorch allocates them); "_host"/plain struct
 *    members are host pointers.  The library copies everything it needs from the host inputs of
 *    chfsi_create during that call; the caller may free them afterwards.  The library owns its device
 *    copies (cell matrices, maps) until chfsi_destroy.
 *  - All device work of the *_dev entry points is enqueued on the caller's cudaStream_t (passed as void*,
 *    NULL = default stream).  They never synchronise the host.  chfsi_create and the *_host entry points
 *    synchronise before returning.
 *  - A handle is NOT re-entrant: it carries mutable state (the spectral shift of the running filter sits on the
 *    diagonals of the stored cell matrices, scratch buffers of the Rayleigh-Ritz products, staging of the *_host
 *    entry point, launch counters).  Host calls on one handle must therefore come from one thread at a time, and
 *    the DEVICE work of successive calls on one handle never overlaps: when a call is enqueued on a different
 *    stream than the previous call on that handle, the library makes the new stream wait (cudaStreamWaitEvent) for
 *    the previous call's work first; the *_host entry point does the same for its internal streams.  Use one handle
 *    per concurrent stream if overlap between filters is wanted.  The caller's workspace belongs to the call that
 *    received it until that call's work has completed.
 *  - There is no CPU fallback: without a CUDA device chfsi_create returns CHFSI_ERR_CUDA.
 *  - Alignment: X_dev / Y_dev / workspace_dev must be 16-byte aligned and B*sizeof(element), ld*sizeof(element)
 *    multiples of 16 (B even for FP64, a multiple of 4 for FP32) for the tensor-core path; other shapes take a
 *    slower generic CUDA path (never the CPU).
 */
#ifndef CHFSI_H_
#define CHFSI_H_

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef enum {
  CHFSI_OK = 0,
  CHFSI_ERR_BAD_ARGUMENT = -1, /* NULL pointer, B < 1, ld < B, m < 1, !(a0 <= a && a < b), bad precision ... */
  CHFSI_ERR_BAD_MESH = -2,     /* dof out of range / repeated inside one cell / non-positive Jacobian         */
  CHFSI_ERR_OUT_OF_MEMORY = -3,
  CHFSI_ERR_CUDA = -4,         /* any CUDA runtime failure, including "no device"                              */
  CHFSI_ERR_UNSUPPORTED = -5   /* p outside 1..8, precision not 32/64                                          */
} chfsi_status;

typedef struct chfsi_op chfsi_op; /* opaque operator handle */

/* Mesh: "cell connectivity, FE degree" (north_star; Sec. 2.3).  All host pointers. */
typedef struct {
  int32_t p;                    /* FE degree 1..8; (p+1)^3 GLL nodes per cell                               */
  int64_t n_cells;
  int64_t n_dofs;
  const int32_t* cell_dofs;     /* [n_cells][(p+1)^3]; local node l = a + (p+1)(b + (p+1)c), x fastest;
                                   periodic identification already applied; dofs distinct inside a cell   */
  const double* cell_vertices;  /* [n_cells][8][3]; vertex v = vx + 2 vy + 4 vz; unwrapped coordinates;
                                   the cell is the trilinear image of [-1,1]^3                             */
} chfsi_mesh;

/* Local potential: V_eff sampled at the (p+2)^3 Gauss-Legendre points of every cell (Eq. 40). */
typedef struct {
  const double* veff_q;         /* [n_cells][(p+2)^3], q = qa + (p+2)(qb + (p+2)qc), x fastest              */
} chfsi_potential;

/* Non-local projectors (Eq. 33).  NULL pointer or n_proj == 0: no such term. */
typedef struct {
  int64_t n_proj;
  const double* D;              /* [n_proj] coupling h_lp (Alg. 4 step 4)                     */
  const int64_t* proj_cell_ptr; /* [n_proj+1] CSR: projector j lives on cells proj_cell_idx[ptr[j]..ptr[j+1]) */
  const int32_t* proj_cell_idx; /* [nnz] cell ids, distinct within one projector                            */
  const double* chi_q;          /* [nnz][(p+2)^3] projector function at the Gauss points of that cell       */
} chfsi_nonlocal;

/* Sizes and the algorithmic work of one H~ application, for benchmarks and tests. */
typedef struct {
  int32_t p, m_cell, n_q, precision, assembly, n_colors;
  int64_t n_cells, n_dofs, n_proj;
  int64_t nnz_cell_proj;        /* sum over cells of N_psp^c (projectors touching the cell)                 */
  int64_t cells_with_proj;
  double flops_per_vector_apply;/* n_cells*2*m_cell^2 + 4*m_cell*nnz_cell_proj + 7*n_dofs  */
  int64_t matrix_bytes;         /* device bytes of the Loewdin-scaled cell matrices (incl. padding)         */
  double sf_flops_per_vector_apply; /* flops the sum-factorised kernel EXECUTES per vector-apply (DMMA at 512
                                   per warp instruction incl. the 7 -> 8 padding, DFMA, projector MMAs of the assembly);
                                   0 when that kernel does not apply to the operator (p > 6)                  */
  int64_t sf_field_bytes;       /* device bytes of its quadrature-point fields and M^-1/2 tables             */
} chfsi_info;

/* assembly: 0 = deterministic (graph colouring of cells that share a dof; every dof is assembled in colour
 *               order -- one launch whose tiles wait on the completion flags of the conflicting earlier cells,
 *               or one launch per colour on the generic path; the recurrence is fused into the first write
 *               of every dof),
 *           1 = atomic (one launch, red.global.add; result depends on summation order within rounding). */
int chfsi_create(chfsi_op** out, const chfsi_mesh* mesh, const chfsi_potential* pot,
                 const chfsi_nonlocal* nl /* nullable */, int precision /* 64 | 32 */,
                 int assembly /* 0 | 1 */, void* cuda_stream);
int chfsi_destroy(chfsi_op* op);

/* k-point variant: the operator that acts on the cell-periodic part u_k of a Bloch wavefunction (Eq. 2-3),
 *   H^k_jl = 1/2 int grad N_j . grad N_l + int (V_eff + 1/2 |k|^2) N_j N_l - i int N_j (k . grad N_l)
 *            + sum_p C^k_pj h_p conj(C^k_pl)                                   (Eq. 30; Eq. 33),
 * complex Hermitian after the Loewdin scaling H~^k = M^-1/2 H^k M^-1/2 (Eq. 34).  The projector samples
 * carry the Bloch phase of Eq. 33: chi_q of `nl` holds the real parts and chi_q_im the imaginary parts of
 *   sum_r e^{-i k.(x - L_r)} chi_p(x, R_a + L_r)  at the Gauss points (same [nnz][(p+2)^3] layout; HOST pointer, copied).
 * A handle made here takes COMPLEX blocks in every block entry point below (chfsi_workspace_bytes, chfsi_apply_H,
 * chfsi_chebyshev_filter, _chunked, _host): element = two FP64 values (re, im), [n_dofs][ld] complex elements with the
 * vector index fastest, B / N / ld counted in complex columns; a0, a, b stay real (the spectrum is real).
 * FE degree p <= 6 and FP64 only (CHFSI_ERR_UNSUPPORTED otherwise); the Rayleigh-Ritz
 * entry points do not take such a handle.  k = 0 with chi_q_im = 0 gives the real operator on both parts. */
typedef struct {
  double k[3];                  /* Bloch wave vector, bohr^-1                                              */
  const double* chi_q_im;       /* [nnz][(p+2)^3]; may be NULL when there are no projectors                */
} chfsi_kpoint;
int chfsi_create_k(chfsi_op** out, const chfsi_mesh* mesh, const chfsi_potential* pot,
                   const chfsi_nonlocal* nl /* nullable */, const chfsi_kpoint* kpoint, int assembly /* 0 | 1 */,
                   void* cuda_stream);

/* New V_eff on the same mesh and projectors: recomputes the Hamiltonian part of every cell matrix,
 *   H^e_jk = 1/2 K^e_jk + sum_q w_q detJ_q V_eff(q) N_j(q) N_k(q)     (Eq. 30 terms 1-2; Eq. 40,
 *   PAPER.md:462-464), Loewdin-scaled (Eq. 34),
 * which is the DHM step of every SCF iteration (Algorithm 1 step 4: V_eff changes with the density).
 * Where the sum-factorised kernel is the operator's default (p <= 6) its operator data are the quadrature-point fields
 * w detJ V_eff(q): the call uploads the samples (kept on the device) and rebuilds those fields in one small kernel; the dense
 * cell matrices are brought up to date from the device copy only when a dense kernel variant is used afterwards.
 * pot->veff_q is a HOST pointer [n_cells][(p+2)^3] (x fastest), copied during the call; projector rows, mesh
 * analysis, colouring and all buffers are reused.  The work is enqueued on cuda_stream and the call returns after
 * synchronising it (the host array may be released).  Must not overlap an apply / filter running on the same
 * handle.  Errors: CHFSI_ERR_BAD_ARGUMENT (NULL), CHFSI_ERR_OUT_OF_MEMORY / CHFSI_ERR_CUDA (temporary buffers). */
int chfsi_update_potential(chfsi_op* op, const chfsi_potential* pot, void* cuda_stream);
int chfsi_get_info(const chfsi_op* op, chfsi_info* info);

/* Device workspace (bytes) that chfsi_apply_H / chfsi_chebyshev_filter need for a block of B columns. */
int chfsi_workspace_bytes(const chfsi_op* op, int64_t B, size_t* bytes);

/* Diagonal GLL mass matrix, FP64, copied to a device array [n_dofs] (for the harness:
 * x~ = M^{1/2} x^). */
int chfsi_mass_diag(const chfsi_op* op, double* M_dev, void* cuda_stream);

/* Y = H~ X for a block of B columns.  X_dev and Y_dev must not overlap. */
int chfsi_apply_H(chfsi_op* op, const void* X_dev, int64_t ldx, void* Y_dev, int64_t ldy, int64_t B,
                  void* workspace_dev, void* cuda_stream);

/* In place: X <- scaled Chebyshev filter of degree m applied to the B columns of X_dev. */
int chfsi_chebyshev_filter(chfsi_op* op, void* X_dev, int64_t ldx, int64_t B, int32_t m, double a, double b,
                           double a0, void* workspace_dev, void* cuda_stream);

/* The same for N columns filtered in sequential chunks of at most B columns ("blocks of B_f
 * vectors filtered sequentially"); workspace sized for B. */
int chfsi_chebyshev_filter_chunked(chfsi_op* op, void* X_dev, int64_t ldx, int64_t N, int64_t B, int32_t m,
                                   double a, double b, double a0, void* workspace_dev, void* cuda_stream);

/* End-to-end variant with HOST buffers: X_host is [n_dofs][ldx] (element type per precision); the call
 * allocates device staging for one chunk, copies each chunk host->device, filters it, copies it back, and
 * synchronises before returning. */
int chfsi_chebyshev_filter_host(chfsi_op* op, void* X_host, int64_t ldx, int64_t N, int64_t B, int32_t m,
                                double a, double b, double a0);

/* Rayleigh-Ritz projection matrices of a (filtered) block Psi_f = Y [n_dofs][ldy], N columns -- Algorithm 2 step 1
 * (RRGEP-OP; the blocked X^T Y products of PAPER.md:556-558), FP64 operators only:
 *   chfsi_overlap_matrix:        S  = Y^T Y                     (step 1a, RRGEP-O)
 *   chfsi_projected_hamiltonian: H^ = Y^T (H~ Y)                (step 1b, RRGEP-P; H~ Y is formed chunk by chunk, B
 *                                                                columns at a time, in the workspace block)
 * S_dev / H_dev are DEVICE arrays [N][N], row-major, FP64, owned by the caller.  N, ldy and B must be even and the
 * pointers 16-byte aligned (CHFSI_ERR_UNSUPPORTED otherwise).  workspace_dev: chfsi_workspace_bytes(op, min(B, N)).
 * Work is enqueued on cuda_stream; the row-split partial sums live in a library-owned scratch buffer that grows on
 * demand (the call then synchronises the stream once).  Both matrices are Hermitian and only their lower triangle is
 * computed (tiles strictly above the diagonal are skipped; for H^ chunk j0 gives the rows >= j0 of its columns);
 * the entries above the diagonal are copies, [r][c] = [c][r], so both triangles are valid and the result is exactly
 * symmetric.  The Cholesky / eigen-decomposition of step 2 is left to the caller (N x N, dense). */
int chfsi_overlap_matrix(chfsi_op* op, const void* Y_dev, int64_t ldy, int64_t N, double* S_dev, void* cuda_stream);
int chfsi_projected_hamiltonian(chfsi_op* op, const void* Y_dev, int64_t ldy, int64_t N, int64_t B, double* H_dev,
                                void* workspace_dev, void* cuda_stream);

/* Allocation-free variant of chfsi_overlap_matrix, for callers that cannot call cudaMalloc (code under CUDA graph capture,
 * tight serving loops, harnesses that forbid it): S = Y^T Y (Algorithm 2 step 1a; lower triangle computed,
 * upper mirrored) with the row-split partial sums in a STATIC device array of the library instead of the
 * scratch buffer that chfsi_overlap_matrix grows on demand.  The call makes no cudaMalloc / cudaFree, creates no event or
 * stream and calls no allocating library routine: it enqueues three kernels on cuda_stream and returns.
 *   limit:   N <= CHFSI_NOALLOC_MAX_N (512) columns; a larger N is CHFSI_ERR_BAD_ARGUMENT with a message that names the
 *            limit.  Any number of rows.  The static array holds CHFSI_NOALLOC_SPLITS x MAX_N x MAX_N doubles = 16 MiB of
 *            device memory on every GPU that loads the library, until the process exits.
 *   sharing: ALL calls on a device (any handle, any stream) use the same array, which keeps the last call's contents;
 *            nothing in it has to start at zero (every partial sum that is read is written by the same call), but two
 *            calls that overlap on the GPU RACE on it: the caller orders them (same stream, or an event between them).
 *            The handle's cross-stream ordering of the other entry points does not cover this call.
 *   device:  the current device must be the one the handle was created on (CHFSI_ERR_CUDA otherwise); the device
 *            address of the array is looked up at chfsi_create*, once per device.
 * Arguments, layout, alignment rules and result as chfsi_overlap_matrix (FP64 operators, real handles; N, ldy even,
 * pointers 16-byte aligned); the sums are split over the rows as there, so the two results agree to rounding (bit for bit
 * when both choose the same number of row splits). */
#define CHFSI_NOALLOC_MAX_N 512
#define CHFSI_NOALLOC_SPLITS 8
int chfsi_overlap_matrix_noalloc(chfsi_op* op, const void* Y_dev, int64_t ldy, int64_t N, double* S_dev, void* cuda_stream);

/* Subspace transformation  Out = Y Z  -- Algorithm 2 step 3 (RRGEP-ST; the blocked "X_p Z"
 * products of PAPER.md:560): with Z = Q_fr it gives the Ritz vectors Psi_fr^R = Psi_f Q_fr (step 3a), with
 * Z = L^-T (S = L L^T) the orthonormal basis Psi^o = Psi_f L^-T (step 3b).  FP64 operators only.
 * Y_dev [n_dofs][ldy] (N columns), Z_dev [N][ldz] (N2 columns, row-major, DEVICE), Out_dev [n_dofs][ldo] (N2
 * columns), all FP64, owned by the caller; Out must not overlap Y (CHFSI_ERR_BAD_ARGUMENT).  N, N2 and the leading
 * dimensions must be even and the pointers 16-byte aligned (CHFSI_ERR_UNSUPPORTED otherwise).  Enqueued on
 * cuda_stream, no synchronisation. */
int chfsi_subspace_transform(chfsi_op* op, const void* Y_dev, int64_t ldy, int64_t N, const double* Z_dev, int64_t ldz,
                             int64_t N2, void* Out_dev, int64_t ldo, void* cuda_stream);

/* Dense N x N step of Algorithm 2 on the device -- step 2a: Cholesky factor S = L L^T and L^-1,
 * which steps 2b (H^ -> L^-1 H^ L^-T) and 3b (Psi^o = Psi_f L^-T) need.  S_dev [N][N] row-major FP64 (symmetric; only
 * the lower triangle is read), L_dev and Linv_dev [N][N] row-major FP64 DEVICE arrays owned by the caller (lower
 * triangular, zeros above the diagonal); info_dev: DEVICE int, 0 on success, else the 1-based index of the first
 * non-positive pivot (S not positive definite: the factors are then meaningless).  Enqueued on cuda_stream, no host
 * synchronisation (the pivot status stays on the device for that reason).  Errors: CHFSI_ERR_BAD_ARGUMENT (NULL, N < 1,
 * N > 16384, overlapping arrays).  The dense symmetric eigenproblem of step 2c is left to the caller (the paper runs it
 * on the CPUs with ELPA). */
int chfsi_cholesky_inverse(chfsi_op* op, const double* S_dev, int64_t N, double* L_dev, double* Linv_dev, int* info_dev,
                           void* cuda_stream);

/* The paper's mixed-precision blocking of the O(M N^2) products of Algorithm 2 (Sec. 3.2; Sec.
 * 4.4.1).  "FP32" blocks: operands rounded to FP32, FP32-level products on the 32-bit tensor pipe (3xTF32
 * split; single-pass TF32 is not used), summed in FP64.  FP64 operators only; N, ldy even; pointers 16-byte aligned;
 * library-owned FP32 copies of the blocks grow on demand (the call then synchronises the stream once).
 *   chfsi_overlap_matrix_mixed:        S = Y^T Y with the diagonal blocks of width `block` in FP64, the rest FP32
 *   chfsi_projected_hamiltonian_mixed: H^ = Y^T (H~ Y) with the split Y = [Y^oc Y^fr] of Eq. 38 (first n_oc columns /
 *                                      the rest): the fr-fr block FP64, the oc-oc, oc-fr and fr-oc blocks FP32 (Eq. 39)
 *   chfsi_subspace_transform_mixed:    Out = SP[Y Z_od] + DP[Y Z_d] for a square Z [N][ldz] (Z = L^-T gives Psi^o,
 *                                      RRGEP-ST-O): off-diagonal entries of Z FP32, diagonal entries FP64
 * Other arguments as in the FP64 calls above; S and H^ are again computed as lower triangles and mirrored (exactly
 * symmetric; the FP32 oc-fr block is the mirror of the fr-oc block). */
int chfsi_overlap_matrix_mixed(chfsi_op* op, const void* Y_dev, int64_t ldy, int64_t N, int64_t block, double* S_dev,
                               void* cuda_stream);
int chfsi_projected_hamiltonian_mixed(chfsi_op* op, const void* Y_dev, int64_t ldy, int64_t N, int64_t B, int64_t n_oc,
                                      double* H_dev, void* workspace_dev, void* cuda_stream);
int chfsi_subspace_transform_mixed(chfsi_op* op, const void* Y_dev, int64_t ldy, int64_t N, const double* Z_dev, int64_t ldz,
                                   void* Out_dev, int64_t ldo, void* cuda_stream);

/* ---- Cell-partitioned operation (the paper's domain decomposition over MPI tasks / GPUs; boundary sums and
 * FP32 boundary traffic; Alg. 4 step 3 across parts) ------------------------------------------
 * A PART is an operator on a subset of the cells of a mesh, with its own dense numbering of the dofs those cells touch.
 * H~ X of the whole mesh is the sum of the parts' results on the dofs they share, provided every part (i) scales with the
 * diagonal mass of the WHOLE mesh and (ii) uses projector coefficients P summed over all parts.  The library gives the pieces;
 * the exchange between the parts (NCCL all-reduce / send-recv) belongs to the caller (paper_2203_07820_b200/partition.py):
 *
 *   chfsi_mesh_mass        host only, no device: diagonal GLL mass M_g = sum_cells w_a w_b w_c detJ of `mesh`
 *                          into mass_host[n_dofs]; a part's partial masses are then summed over the parts by the caller.
 *   chfsi_create_part      chfsi_create with the mass of the whole mesh at the part's dofs given (dof_mass[n_dofs], HOST).
 *   chfsi_projector_coefficients      steps 3a-3c of the path on the part's cells: P_dev[n_proj][B] (operator's storage type,
 *                          vector index fastest) = D (C^T X) restricted to the part's cells; summing it over the parts gives P.
 *   chfsi_apply_H_with_coefficients   chfsi_apply_H with steps 3a-3c replaced by the given P_dev[n_proj][B]: Y = the part's
 *                          contribution to H~ X (complete on interior dofs, partial on shared ones).
 *   chfsi_pack_rows / chfsi_unpack_rows   buf[s(i)][0..B) = X[rows[i]][0..B) and back, s(i) = slots_dev[i] (or i when slots_dev is
 *                          NULL; the slots let every part write into one buffer laid out over all shared dofs); buf is a
 *                          dense [.][B] array; buf_precision = the operator's precision, or 32 for the paper's FP32
 *                          boundary payload; X is any [rows][ld] block of the operator's type; rows_dev / slots_dev are
 *                          DEVICE int32 arrays.
 *   chfsi_recurrence_update            T <- alpha (HX - c X) - beta T on whole blocks: one degree of the scaled recurrence
 *                          (Eq. 37) once HX is complete on every dof.
 * All device work is enqueued on the stream; same block conventions and error codes as above.  Not for k-point handles. */
int chfsi_mesh_mass(const chfsi_mesh* mesh, double* mass_host);
int chfsi_create_part(chfsi_op** out, const chfsi_mesh* mesh, const chfsi_potential* pot, const chfsi_nonlocal* nl /* nullable */,
                      const double* dof_mass, int precision /* 64 | 32 */, int assembly /* 0 | 1 */, void* cuda_stream);
int chfsi_projector_coefficients(chfsi_op* op, const void* X_dev, int64_t ldx, int64_t B, void* P_dev, void* workspace_dev,
                                 void* cuda_stream);
int chfsi_apply_H_with_coefficients(chfsi_op* op, const void* X_dev, int64_t ldx, void* Y_dev, int64_t ldy, int64_t B,
                                    const void* P_dev, void* workspace_dev, void* cuda_stream);
int chfsi_pack_rows(chfsi_op* op, const void* X_dev, int64_t ldx, int64_t B, const int32_t* rows_dev,
                    const int32_t* slots_dev /* nullable */, int64_t n_rows, void* buf_dev, int buf_precision, void* cuda_stream);
int chfsi_unpack_rows(chfsi_op* op, const void* buf_dev, int buf_precision, const int32_t* rows_dev,
                      const int32_t* slots_dev /* nullable */, int64_t n_rows, void* X_dev, int64_t ldx, int64_t B,
                      void* cuda_stream);
int chfsi_recurrence_update(chfsi_op* op, const void* HX_dev, int64_t ldh, const void* X_dev, int64_t ldx, void* T_dev,
                            int64_t ldt, int64_t B, double alpha, double beta, double c, void* cuda_stream);

/* The same exchange for the filter in SCALED blocks (the accumulate-only recurrence W_k = W_{k-2} + gamma_k (H~ - c) W_{k-1} of
 * chfsi_chebyshev_filter, U14), which saves the separate recurrence pass over the block: the part's cell kernel adds
 * its contribution straight into the block that holds W_{k-2}, and only the rows of the shared dofs are fixed up afterwards.
 *   chfsi_accumulate_supported   *supported = 1 when chfsi_apply_shifted_with_coefficients can ADD for these blocks (the
 *                          sum-factorised kernel: p <= 6, kernel variant 0 or 6, 16-byte aligned blocks); else 0 and the caller
 *                          stays with chfsi_apply_H_with_coefficients + chfsi_recurrence_update.  No device work.
 *   chfsi_apply_shifted_with_coefficients   T = alpha (H~_part - c) X  (accumulate = 0: the part's first contribution to a dof is
 *                          a store, T need not be initialised) or  T += alpha (H~_part - c) X  (accumulate = 1;
 *                          CHFSI_ERR_UNSUPPORTED where chfsi_accumulate_supported says 0), projector coefficients P_dev given.
 *                          EVERY part subtracts c X once on each dof it holds, shared or not.
 *   chfsi_pack_rows_delta  buf[s(i)] = T[rows[i]] - base[i] + corr X[rows[i]] (1 - owner[i]): the part's contribution to its
 *                          shared rows.  base_dev [n_rows][B] (dense, operator's type) = those rows of T as packed by
 *                          chfsi_pack_rows BEFORE the accumulating application (NULL after a storing one: 0); owner_dev[n_rows]
 *                          (DEVICE bytes) = 1 on the one part that owns the dof, 0 on the others, which put the shift back:
 *                          corr = alpha c.  Summed over the parts, buf is alpha (H~ - c) X on the shared dofs.
 *   chfsi_unpack_rows_sum  T[rows[i]] = base[i] + buf[s(i)]  (base_dev NULL: 0), the sums back in place.
 * buf, slots, precisions and error codes as in chfsi_pack_rows / chfsi_unpack_rows. */
int chfsi_accumulate_supported(chfsi_op* op, const void* X_dev, int64_t ldx, const void* T_dev, int64_t ldt, int64_t B,
                               void* workspace_dev, int* supported);
int chfsi_apply_shifted_with_coefficients(chfsi_op* op, const void* X_dev, int64_t ldx, void* T_dev, int64_t ldt, int64_t B,
                                          double alpha, double c, int accumulate, const void* P_dev, void* workspace_dev,
                                          void* cuda_stream);
int chfsi_pack_rows_delta(chfsi_op* op, const void* T_dev, int64_t ldt, const void* base_dev /* nullable */, const void* X_dev,
                          int64_t ldx, const uint8_t* owner_dev, double corr, int64_t B, const int32_t* rows_dev,
                          const int32_t* slots_dev /* nullable */, int64_t n_rows, void* buf_dev, int buf_precision,
                          void* cuda_stream);
int chfsi_unpack_rows_sum(chfsi_op* op, const void* buf_dev, int buf_precision, const void* base_dev /* nullable */,
                          const int32_t* rows_dev, const int32_t* slots_dev /* nullable */, int64_t n_rows, void* T_dev,
                          int64_t ldt, int64_t B, void* cuda_stream);

/* Number of kernel launches enqueued by this handle since creation (for benchmark bookkeeping). */
int64_t chfsi_launch_count(const chfsi_op* op);

/* Selects the kernel used for the per-cell product H~^e X^e (all variants compute the same H~ X up to rounding):
 *   0 = automatic: the warp-specialised sum-factorised (matrix-free) kernel for FE degree p <= 6 (north_star:
 *       "sum-factorised where measurement says so"; csrc/apply_sf_ws.cuh; a three-term update with beta != 0 asked for
 *       outside chfsi_chebyshev_filter goes to the kernel of variant 5), else the dense persistent tensor-core kernel,
 *       else the generic path;
 *   1 = generic dense path (any shape / alignment);
 *   2 = dense tensor-core kernel, one launch per colour;
 *   3 = (FP32 storage only) dense, 3xTF32 products on the 32-bit tensor pipe: outside the 1e-5 Ha eigenvalue
 *       tolerance of the FP32 variant (csrc/apply_tf32.cuh);
 *   4 = dense persistent tensor-core kernel (FP64 DMMA with the distinct per-cell matrices of Eq. 47);
 *   5 = sum-factorised kernel, one CTA = column loop + tile hand-over (csrc/apply_sf.cuh; the round-2 predecessor of 6);
 *   6 = warp-specialised sum-factorised kernel (same as 0 where it applies): the filter runs its recurrence in scaled
 *       blocks so that every contribution to the target block is an addition (csrc/api.cu filter_block).
 * For tests and A/B measurements. */
int chfsi_set_kernel_variant(chfsi_op* op, int variant);

/* Kernel of the FP32 blocks of the mixed-precision Rayleigh-Ritz products S and H^ (3xTF32 products, FP64 totals):
 *   0 = automatic = 1;  1 = tcgen05.mma kind::tf32 with TMEM accumulators, operands by TMA (csrc/rr_umma.cu);
 *   2 = mma.sync m16n8k8 (csrc/rr_kernels.cu k_xty_tf32).  Same results up to the rounding of the FP32 partial sums. */
int chfsi_set_rr_variant(chfsi_op* op, int variant);

/* Per-kernel device timing for the roofline report.  While enabled, every H~ application records one CUDA
 * event pair on the launching stream around its per-cell contraction launches (the dominant kernel; steps 1,
 * 2, 3d, 4, 5 of the path) and one around its projector launches (steps 3a-3c).  chfsi_get_profile waits for
 * the recorded events, returns the accumulated device time and launch counts since profiling was enabled (or
 * last read), and resets the accumulators. */
typedef struct {
  double contraction_ms;        /* summed device time of the contraction launches                           */
  int64_t contraction_launches; /* number of those launches (one per colour, or one in atomic mode)          */
  double projector_ms;          /* summed device time of the projector launches (incl. atomic-mode pre-fill) */
  int64_t projector_launches;
  int64_t applies;              /* H~ applications covered                                                   */
} chfsi_profile;
int chfsi_set_profiling(chfsi_op* op, int enabled);
int chfsi_get_profile(chfsi_op* op, chfsi_profile* prof);

/* FP64 peak of the current device in TFLOP/s, measured with register-resident loops of mma.sync m8n8k4 f64
 * (the tensor pipe used by the per-cell contraction) and of plain DFMA; best of 5 launches of ~10 ms each.
 * This is the roofline denominator of the contraction kernel (MEASURED_PEAKS.json has no FP64 figure).
 * Synchronises the host. */
int chfsi_measure_fp64_peak(double* dmma_tflops, double* dfma_tflops, void* cuda_stream);

const char* chfsi_last_error(const chfsi_op* op /* NULL: last failed chfsi_create of this thread */);

#ifdef __cplusplus
}
#endif
#endif /* CHFSI_H_ */
