// Hot-path kernels of libchfsi: one fused launch sequence per H~ application + Chebyshev recurrence update.
//
//   step 1  cell extraction          X^e = rows of X through the cell->dof map      PAPER.md:513 (i), :515
//   step 2  per-cell contraction     Y^e = H~^e X^e    (FP64: mma.sync m8n8k4 DMMA)   Eq. 47
//   step 3  non-local                P^c = C~^cT X^e ; P = D sum_c P^c ; Y^e += C~^c P   Alg. 4
//   step 4  assembly                 T[g] += Y^e[l]    (coloured or atomic)           PAPER.md:513 (iii)
//   step 5  recurrence               Y_k = alpha (H~ Y_{k-1} - c Y_{k-1}) - beta Y_{k-2}   Eq. 37
//
// Steps 1, 2, 3d (as extra contraction rows), 4 and 5 run inside ONE kernel (k_apply_dmma / k_apply_generic);
// steps 3a-3c are two small kernels in front of it because P needs every cell of a projector's support.
// M^-1/2 is folded into the cell matrices at setup, so no scaling appears here.
#include <algorithm>
#include <cstdio>
#include <cstdlib>

#include <cuda.h>   // CUtensorMap (types only; the encoder is fetched through cudaGetDriverEntryPoint)

#include "common.h"

namespace chfsi {

namespace {

template <typename T>
struct ApplyDev {
  const T* __restrict__ mat;
  const int64_t* __restrict__ mat_off;
  const int64_t* __restrict__ idx_off;
  const int32_t* __restrict__ ktot;
  const int32_t* __restrict__ gidx;
  const int32_t* __restrict__ cells;   // cells of this launch
  int n_launch_cells;
  int n_col_tiles;
  int m_cell, mpad, lda;               // mpad = round8(m_cell): projector rows of the contraction start there
  int mw, n_parts;                     // output columns per matrix block / blocks per cell (common.h, Op::n_parts)
  const T* __restrict__ X; int64_t ldx;
  T* __restrict__ Tg; int64_t ldt;
  const T* __restrict__ P; int64_t ldp;
  int B;
  T alpha, beta;                       // T <- alpha (H~ - c) X - beta T ; the shift c sits on the matrix diagonals
  int atomic;                          // 1: red.add into a pre-filled target
  int accumulate;                      // 1: T <- T + alpha (H~ - c) X (k_apply_sf_ws; common.h ApplyArgs::accumulate)
};

__device__ __forceinline__ void red_add(double* p, double v) { atomicAdd(p, v); }
__device__ __forceinline__ void red_add(float* p, float v) { atomicAdd(p, v); }

// -------------------------------------------------------------------------------------------------------------
// Generic path: any B, any alignment, any p, double or float.  One CTA = (cell, 32 columns); lane = column.
// -------------------------------------------------------------------------------------------------------------
template <typename T>
__global__ void __launch_bounds__(256) k_apply_generic(ApplyDev<T> a) {
  extern __shared__ __align__(128) unsigned char smem_raw[];
  T* Xs = reinterpret_cast<T*>(smem_raw);          // [kt][32]
  const int cell = a.cells[blockIdx.x / a.n_col_tiles];
  const int col = (blockIdx.x % a.n_col_tiles) * 32 + (threadIdx.x & 31);
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  const int kt = a.ktot[cell], mc = a.m_cell;
  const int32_t* gi = a.gidx + a.idx_off[cell];
  const T* M = a.mat + a.mat_off[cell];
  const bool colok = col < a.B;
  for (int k = warp; k < kt; k += 8) {
    int idx = gi[k];
    const T* src = (k < a.mpad) ? a.X + (int64_t)(idx & 0x7fffffff) * a.ldx : a.P + (int64_t)idx * a.ldp;
    Xs[k * 32 + lane] = colok ? src[col] : (T)0;
  }
  __syncthreads();
  const int n_rt = (mc + 7) / 8;
  for (int rt = warp; rt < n_rt; rt += 8) {
    T acc[8];
#pragma unroll
    for (int i = 0; i < 8; ++i) acc[i] = (T)0;
    const T* Mr = M + mat_elem(0, rt * 8, a.mw, a.lda, kt);   // the 8 rows of an output tile sit in one block
    for (int k = 0; k < kt; ++k) {
      T x = Xs[k * 32 + lane];
#pragma unroll
      for (int i = 0; i < 8; ++i) acc[i] = fma(Mr[(int64_t)k * a.lda + i], x, acc[i]);
    }
    if (!colok) continue;
#pragma unroll
    for (int i = 0; i < 8; ++i) {
      int r = rt * 8 + i;
      if (r >= mc) break;
      int idx = gi[r];
      int64_t g = idx & 0x7fffffff;
      T* tp = a.Tg + g * a.ldt + col;
      T v = a.alpha * acc[i];
      if (a.atomic) {
        red_add(tp, v);
      } else if (idx < 0) {   // first contribution to this dof: carries the recurrence term -beta Y_{k-2}
        if (a.beta != (T)0) v = fma(-a.beta, *tp, v);
        *tp = v;
      } else {
        *tp += v;
      }
    }
  }
}

// -------------------------------------------------------------------------------------------------------------
// Steps 3a-3c.  Alg. 4 steps 2-3 compute P = sum_c C^cT X^c cell by cell and assemble over the cells of each
// projector.  C is constant, so that assembly is applied to C once at setup
// (assemble_projector_rows: coefficient of dof g = s_g sum_{c containing g} C^c[l(g)][j]) and per apply
// P[j] = sum_g coef[g][j] X[g]: every dof row of X in the support of an atom is read ONCE (not once per cell) for
// all of the atom's <= 8 projectors.  HBM-bound row stream.
// -------------------------------------------------------------------------------------------------------------
// grid = (row segments of <= 128 dofs) x (256-column tiles); thread = (row slot rs = tid/128, 2 columns): a row is
// read as 128 x 16-byte pieces (coalesced), its 8 coefficients come from shared memory (broadcast), the two row
// slots are summed in slot order through shared memory: deterministic.  64 registers -> 4 CTAs/SM with 8 rows in
// flight per thread: the kernel lives on memory-level parallelism.  Partial sums are FP64 for both precisions.
constexpr int kPRCols = 256;
template <typename T>
__global__ void __launch_bounds__(256, 4) k_proj_rows(const int32_t* __restrict__ seg_ptr, const int32_t* __restrict__ grow_dof,
                                                      const T* __restrict__ pcoef, const T* __restrict__ X, int64_t ldx,
                                                      double* __restrict__ Pc, int B, int vec_ok) {
  __shared__ double red[kProjGroup][kPRCols];
  __shared__ __align__(16) T cs[kProjSegRows * kProjGroup];
  __shared__ int32_t dofs[kProjSegRows];
  const int seg = blockIdx.x;
  const int r0 = seg_ptr[seg], nr = seg_ptr[seg + 1] - r0;
  const int tid = threadIdx.x, cg = tid & 127, rs = tid >> 7;
  const int col = blockIdx.y * kPRCols + cg * 2;
  for (int e = tid; e < nr * kProjGroup; e += 256) cs[e] = pcoef[(int64_t)r0 * kProjGroup + e];
  for (int e = tid; e < nr; e += 256) dofs[e] = grow_dof[r0 + e];
  __syncthreads();
  double acc[kProjGroup][2];
#pragma unroll
  for (int i = 0; i < kProjGroup; ++i) acc[i][0] = acc[i][1] = 0.0;
  const bool full2 = vec_ok && (col + 1 < B);
  if (col < B) {
#pragma unroll 8
    for (int r = rs; r < nr; r += 2) {
      const T* xr = X + (int64_t)dofs[r] * ldx + col;
      double x0, x1;
      if (full2) {
        if constexpr (sizeof(T) == 8) {
          const double2 u = *reinterpret_cast<const double2*>(xr);
          x0 = u.x; x1 = u.y;
        } else {
          const float2 u = *reinterpret_cast<const float2*>(xr);
          x0 = u.x; x1 = u.y;
        }
      } else {
        x0 = (double)xr[0]; x1 = (col + 1 < B) ? (double)xr[1] : 0.0;
      }
#pragma unroll
      for (int i = 0; i < kProjGroup; ++i) {
        const double c = (double)cs[r * kProjGroup + i];
        acc[i][0] = fma(c, x0, acc[i][0]);
        acc[i][1] = fma(c, x1, acc[i][1]);
      }
    }
  }
  if (rs == 1) {
#pragma unroll
    for (int i = 0; i < kProjGroup; ++i) { red[i][cg * 2] = acc[i][0]; red[i][cg * 2 + 1] = acc[i][1]; }
  }
  __syncthreads();
  if (rs == 0 && col < B) {
#pragma unroll
    for (int i = 0; i < kProjGroup; ++i) {
      double* out = Pc + ((int64_t)seg * kProjGroup + i) * B + col;
      out[0] = acc[i][0] + red[i][cg * 2];
      if (col + 1 < B) out[1] = acc[i][1] + red[i][cg * 2 + 1];
    }
  }
}

// P[j][col] = D_j sum_{segments of j's group} Pc[seg][slot_j][col], segment order (Alg. 4 step 4 is the D scaling,
// PAPER.md:527); row n_proj = 0 (target of the padding rows of the contraction)
template <typename T>
__global__ void __launch_bounds__(128) k_proj_reduce(const double* __restrict__ Pc, const int32_t* __restrict__ grp_seg_ptr,
                                                     const int32_t* __restrict__ proj_grp, const int32_t* __restrict__ proj_slot,
                                                     const double* __restrict__ D, int64_t n_proj, T* __restrict__ P, int B) {
  const int64_t j = blockIdx.x;
  const int col = blockIdx.y * 128 + threadIdx.x;
  if (col >= B) return;
  double s = 0.0;
  if (j < n_proj && proj_grp[j] >= 0) {
    const int g = proj_grp[j], slot = proj_slot[j];
    for (int seg = grp_seg_ptr[g]; seg < grp_seg_ptr[g + 1]; ++seg) s += Pc[((int64_t)seg * kProjGroup + slot) * B + col];
    s *= D[j];
  }
  P[j * B + col] = (T)s;
}

// setup: projector rows of the cell matrices -> compact FP64 rows [nnz_cp][m_cell]
template <typename T>
__global__ void __launch_bounds__(128) k_extract_proj_rows(const T* __restrict__ mat, const int64_t* __restrict__ mat_off,
                                                           const int64_t* __restrict__ cell_proj_ptr,
                                                           const int32_t* __restrict__ row_cell,
                                                           const int32_t* __restrict__ ktot, int m_cell, int mpad, int lda,
                                                           int mw, double* __restrict__ out /*[rows][mpad]*/) {
  const int64_t r = blockIdx.x;
  const int c = row_cell[r];
  const int krow = mpad + (int)(r - cell_proj_ptr[c]);
  const T* M = mat + mat_off[c];
  for (int l = threadIdx.x; l < mpad; l += 128) out[r * mpad + l] = l < m_cell ? (double)M[mat_elem(krow, l, mw, lda, ktot[c])] : 0.0;
}

// Atomic assembly needs the recurrence term in place first:  T <- -beta T
template <typename T>
__global__ void __launch_bounds__(256) k_prefill(T* __restrict__ Tg, int64_t ldt, int64_t n_dofs, int B, T beta) {
  int64_t n = n_dofs * B;
  for (int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (int64_t)gridDim.x * blockDim.x) {
    int64_t g = i / B; int col = (int)(i % B);
    T v = (T)0;
    if (beta != (T)0) v = -beta * Tg[g * ldt + col];
    Tg[g * ldt + col] = v;
  }
}

// The spectral shift c of the filter lives on the diagonals of the cell matrices (common.h, Op::diag0): the
// (cell, node) that makes the first contribution to a dof carries -c for that dof.
template <typename T>
__global__ void __launch_bounds__(256) k_set_diag_shift(T* __restrict__ mat, const int64_t* __restrict__ mat_off,
                                                        const int64_t* __restrict__ idx_off, const int32_t* __restrict__ gidx,
                                                        const int32_t* __restrict__ ktot, const double* __restrict__ diag0,
                                                        int m_cell, int lda, int mw, int64_t n_cells, double shift) {
  const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= n_cells * m_cell) return;
  const int64_t c = i / m_cell;
  const int k = (int)(i - c * m_cell);
  const bool first = gidx[idx_off[c] + k] < 0;
  mat[mat_off[c] + mat_elem(k, k, mw, lda, ktot[c])] = (T)(diag0[i] - (first ? shift : 0.0));
}
template <typename T>
__global__ void __launch_bounds__(256) k_capture_diag(const T* __restrict__ mat, const int64_t* __restrict__ mat_off,
                                                      const int32_t* __restrict__ ktot, double* __restrict__ diag0,
                                                      int m_cell, int lda, int mw, int64_t n_cells) {
  const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= n_cells * m_cell) return;
  const int64_t c = i / m_cell;
  const int k = (int)(i - c * m_cell);
  diag0[i] = (double)mat[mat_off[c] + mat_elem(k, k, mw, lda, ktot[c])];
}

// -------------------------------------------------------------------------------------------------------------
// Tensor-core path (FP64): CTA = (cell, 64 columns), 16 warps as 4 (m) x 4 (n); warp tile = MT m-tiles x 2 n-tiles
// of mma.sync.m8n8k4.f64.  The cell matrix is streamed in 16-row K-panels by cp.async.bulk (one bulk copy per
// panel; the HBM image of the matrix IS the padded shared-memory image), X^e rows are gathered by one bulk copy per
// row through the cell->dof map, both landing on an mbarrier; 3-stage ring.
// -------------------------------------------------------------------------------------------------------------
constexpr int kPanelK = 16;
constexpr int kTileN = 64;
constexpr int kLdXs = kTileN + 4;    // 68: 68 mod 16 == 4 -> conflict-free 64-bit fragment loads
constexpr int kStages = 3;
constexpr int kMaxKtot = 1024;

__device__ __forceinline__ uint32_t smem_u32(const void* p) { return (uint32_t)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void mbar_init(uint64_t* bar, int count) {
  asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(bar)), "r"(count));
}
__device__ __forceinline__ void mbar_expect_tx(uint64_t* bar, uint32_t bytes) {
  asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(bar)), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_wait(uint64_t* bar, uint32_t parity) {
  uint32_t done;
  do {
    asm volatile(
        "{\n"
        ".reg .pred p;\n"
        "mbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n"
        "selp.u32 %0, 1, 0, p;\n"
        "}\n"
        : "=r"(done)
        : "r"(smem_u32(bar)), "r"(parity)
        : "memory");
  } while (!done);
}
__device__ __forceinline__ void bulk_g2s(void* dst, const void* src, uint32_t bytes, uint64_t* bar) {
  asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];" ::"r"(smem_u32(dst)),
               "l"(src), "r"(bytes), "r"(smem_u32(bar))
               : "memory");
}
__device__ __forceinline__ void dmma884(double& c0, double& c1, double a, double b) {
  asm("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1}, {%2}, {%3}, {%0,%1};" : "+d"(c0), "+d"(c1) : "d"(a), "d"(b));
}

template <int MT>
__global__ void __launch_bounds__(512, 1) k_apply_dmma(ApplyDev<double> a) {
  extern __shared__ __align__(128) unsigned char smem_raw[];
  const int lda = a.lda;
  const int a_panel_elems = kPanelK * lda;
  const int stage_elems = a_panel_elems + kPanelK * kLdXs;
  double* stage0 = reinterpret_cast<double*>(smem_raw);
  uint64_t* full = reinterpret_cast<uint64_t*>(stage0 + kStages * stage_elems);
  int32_t* idx_s = reinterpret_cast<int32_t*>(full + kStages);

  const int cell = a.cells[blockIdx.x / a.n_col_tiles];
  const int col0 = (blockIdx.x % a.n_col_tiles) * kTileN;
  const int ncols = min(kTileN, a.B - col0);             // multiple of 8
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  const int warp_m = warp >> 2, warp_n = warp & 3;
  const int kt = a.ktot[cell], mc = a.m_cell;
  const int32_t* gi = a.gidx + a.idx_off[cell];
  const double* M = a.mat + a.mat_off[cell];

  for (int k = tid; k < kt; k += 512) idx_s[k] = gi[k];
  if (tid == 0) {
    for (int s = 0; s < kStages; ++s) mbar_init(&full[s], 1);
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
  }
  __syncthreads();

  const int npanel = (kt + kPanelK - 1) / kPanelK;
  const uint32_t row_bytes = (uint32_t)ncols * 8u;
  auto issue = [&](int pi) {   // called by warp 0, all lanes
    const int s = pi % kStages;
    const int rows = min(kPanelK, kt - pi * kPanelK);
    double* As = stage0 + s * stage_elems;
    double* Xs = As + a_panel_elems;
    if (lane == 0) mbar_expect_tx(&full[s], (uint32_t)rows * ((uint32_t)lda * 8u + row_bytes));
    __syncwarp();
    if (lane < rows) {
      const int k = pi * kPanelK + lane;
      const int idx = idx_s[k];
      const double* src = (k < a.mpad) ? a.X + (int64_t)(idx & 0x7fffffff) * a.ldx + col0 : a.P + (int64_t)idx * a.ldp + col0;
      bulk_g2s(Xs + lane * kLdXs, src, row_bytes, &full[s]);
    } else if (lane == 16) {
      bulk_g2s(As, M + (int64_t)pi * a_panel_elems, (uint32_t)rows * (uint32_t)lda * 8u, &full[s]);
    }
  };
  if (warp == 0)
    for (int pi = 0; pi < kStages - 1 && pi < npanel; ++pi) issue(pi);

  // warp tile
  const int n_mtiles = (mc + 7) / 8;
  const int mt0 = warp_m * MT;
  const int nmt = max(0, min(MT, n_mtiles - mt0));
  const int nt0 = warp_n * 2;
  const int nnt = max(0, min(2, ncols / 8 - nt0));
  double acc[MT][2][2];
#pragma unroll
  for (int i = 0; i < MT; ++i)
#pragma unroll
    for (int j = 0; j < 2; ++j) acc[i][j][0] = acc[i][j][1] = 0.0;

  const int fk = lane & 3, fm = lane >> 2;
  for (int pi = 0; pi < npanel; ++pi) {
    const int s = pi % kStages;
    mbar_wait(&full[s], (uint32_t)((pi / kStages) & 1));
    __syncthreads();   // every warp is done with panel pi-1: its ring slot may be refilled
    if (warp == 0 && pi + kStages - 1 < npanel) issue(pi + kStages - 1);
    if (nnt == 0 || nmt == 0) continue;
    const double* As = stage0 + s * stage_elems;
    const double* Xs = As + a_panel_elems;
    const int ksteps = min(kPanelK, kt - pi * kPanelK) / 4;
    const double* Ap = As + fk * lda + mt0 * 8 + fm;
    const double* Xp = Xs + fk * kLdXs + nt0 * 8 + fm;
    for (int ks = 0; ks < ksteps; ++ks) {
      double b0 = Xp[0], b1 = (nnt > 1) ? Xp[8] : 0.0;
#pragma unroll
      for (int i = 0; i < MT; ++i) {
        if (i < nmt) {
          double av = Ap[i * 8];
          dmma884(acc[i][0][0], acc[i][0][1], av, b0);
          dmma884(acc[i][1][0], acc[i][1][1], av, b1);
        }
      }
      Ap += 4 * lda;
      Xp += 4 * kLdXs;
    }
  }

  // epilogue: assembly + recurrence (steps 4-5).  C fragment: row = lane/4, columns 2*(lane%4) + {0,1}
  const double alpha = a.alpha, beta = a.beta;
#pragma unroll
  for (int i = 0; i < MT; ++i) {
    if (i >= nmt) continue;
    const int r = (mt0 + i) * 8 + fm;
    if (r >= mc) continue;
    const int idx = idx_s[r];
    const int64_t g = idx & 0x7fffffff;
#pragma unroll
    for (int j = 0; j < 2; ++j) {
      if (j >= nnt) continue;
      const int col = col0 + (nt0 + j) * 8 + fk * 2;
      double2* tp = reinterpret_cast<double2*>(a.Tg + g * a.ldt + col);
      double v0 = alpha * acc[i][j][0], v1 = alpha * acc[i][j][1];
      if (a.atomic) {
        atomicAdd(&tp->x, v0);
        atomicAdd(&tp->y, v1);
      } else if (idx < 0) {
        if (beta != 0.0) {
          double2 t = *tp;
          v0 = fma(-beta, t.x, v0); v1 = fma(-beta, t.y, v1);
        }
        *tp = make_double2(v0, v1);
      } else {
        double2 t = *tp;
        *tp = make_double2(t.x + v0, t.y + v1);
      }
    }
  }
}


// -------------------------------------------------------------------------------------------------------------
// Tensor-core path v2 (FP64, default): ONE persistent launch per H~ application.
//   tile   = (cell, 32 columns); 8 warps as 4 (m) x 2 (n), warp tile = MT m-tiles x 2 n-tiles of m8n8k4 DMMA;
//            two CTAs per SM, so one CTA's prologue / epilogue runs under the other's main loop.
//   order  = tiles are handed out by an atomic ticket in (colour, cell, column tile) order.  A tile's epilogue
//            waits for the completion flags of the earlier cells that share a dof with its cell (same column
//            tile only), so every dof is assembled in colour order -> bit-reproducible, with no launch boundary
//            and no wave tail between colours.  A ticket holder only ever waits on lower tickets, all of which
//            are held by running CTAs: no deadlock.
//   stream = 8-row K-panels of the cell matrix (one bulk copy, UBLKCP) + the 8 matching rows of X gathered through
//            the cell->dof map by two TMA row gathers (cp.async.bulk.tensor.2d.tile::gather4, UTMALDG.2D.GATHER4:
//            four arbitrary rows of the [n_dofs x B] block per instruction) land on a "full" mbarrier of a
//            4-stage ring; ONE lane issues the three copies of a panel, nobody touches the data on the way;
//            warps release a stage through an "empty" mbarrier as soon as their fragments are in registers.
// -------------------------------------------------------------------------------------------------------------
constexpr int kP2PanelK = 8;
constexpr int kP2TileN = 32;
constexpr int kP2LdXs = kP2TileN;       // the TMA row gather packs the rows densely (256 B each)
constexpr int kP2Threads = 256;
// ring depth: 4 stages of 24 KB for FP64 storage, 8 stages of 12 KB for FP32 storage; panels in flight = stages - 2
// (one slot of slack so that a producer never waits for the previous producer, which lags by its own issue time)
template <typename S> __host__ __device__ constexpr int p2_stages() { return sizeof(S) == 8 ? 4 : 8; }
constexpr int kSyncFlagOffset = 32;     // uint32 index of the first flag inside the sync region (128 bytes)

struct PersistDev {
  const int32_t* __restrict__ pos_cell;    // cell at position t of the colour order
  const int32_t* __restrict__ dep_ptr;
  const int32_t* __restrict__ dep_pos;
  unsigned long long* counter;
  uint32_t* flags;                          // [n_cells][n_col_tiles]
  unsigned long long ticket_base;
  uint32_t epoch;
  int n_tiles;
};

__device__ __forceinline__ void mbar_arrive(uint64_t* bar) {
  asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(smem_u32(bar)) : "memory");
}
// four rows r0..r3 of a 2-D tensor (columns c0 .. c0+box-1) -> four consecutive box-wide rows at dst
__device__ __forceinline__ void tma_gather4(void* dst, const CUtensorMap* tm, int c0, int r0, int r1, int r2, int r3,
                                            uint64_t* bar) {
  asm volatile(
      "cp.async.bulk.tensor.2d.shared::cluster.global.tile::gather4.mbarrier::complete_tx::bytes [%0], [%1, {%3, %4, %5, %6, %7}], [%2];"
      ::"r"(smem_u32(dst)), "l"(tm), "r"(smem_u32(bar)), "r"(c0), "r"(r0), "r"(r1), "r"(r2), "r"(r3)
      : "memory");
}
__device__ __forceinline__ uint32_t ld_acquire_gpu(const uint32_t* p) {
  uint32_t v;
  asm volatile("ld.acquire.gpu.global.u32 %0, [%1];" : "=r"(v) : "l"(p) : "memory");
  return v;
}
__device__ __forceinline__ void st_release_gpu(uint32_t* p, uint32_t v) {
  asm volatile("st.release.gpu.global.u32 [%0], %1;" ::"l"(p), "r"(v) : "memory");
}
__device__ __forceinline__ double2 ld_cg_d2(const double* p) {
  double2 v;
  asm volatile("ld.global.cg.v2.f64 {%0,%1}, [%2];" : "=d"(v.x), "=d"(v.y) : "l"(p) : "memory");
  return v;
}

__device__ __forceinline__ double2 ld_cg_pair(const double* p) { return ld_cg_d2(p); }
__device__ __forceinline__ double2 ld_cg_pair(const float* p) {
  float x, y;
  asm volatile("ld.global.cg.v2.f32 {%0,%1}, [%2];" : "=f"(x), "=f"(y) : "l"(p) : "memory");
  return make_double2((double)x, (double)y);
}
__device__ __forceinline__ void st_pair(double* p, double v0, double v1) { *reinterpret_cast<double2*>(p) = make_double2(v0, v1); }
__device__ __forceinline__ void st_pair(float* p, double v0, double v1) { *reinterpret_cast<float2*>(p) = make_float2((float)v0, (float)v1); }

// S = storage type of the cell matrices and the vector blocks (double, or float for the FP32 variant: the fragments
// are widened to FP64 in registers and the contraction still runs on the FP64 tensor pipe with FP64 accumulators).
template <int MT, typename S>
__global__ void __launch_bounds__(kP2Threads, 2) k_apply_dmma_p(ApplyDev<S> a, PersistDev pd,
                                                                const __grid_constant__ CUtensorMap tmX,
                                                                const __grid_constant__ CUtensorMap tmP) {
  extern __shared__ __align__(128) unsigned char smem_raw[];
  const int lda = a.lda;
  const int a_panel_elems = kP2PanelK * lda;
  const int stage_elems = a_panel_elems + kP2PanelK * kP2LdXs;
  constexpr int kP2Stages = p2_stages<S>();
  constexpr int kP2Ahead = kP2Stages - 2;
  S* stage0 = reinterpret_cast<S*>(smem_raw);
  uint64_t* full = reinterpret_cast<uint64_t*>(stage0 + kP2Stages * stage_elems);
  uint64_t* empty = full + kP2Stages;
  long long* ticket_s = reinterpret_cast<long long*>(empty + kP2Stages);   // [2]
  int32_t* idx_s = reinterpret_cast<int32_t*>(ticket_s + 2);

  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  const int warp_m = warp >> 1, warp_n = warp & 1;
  const int fk = lane & 3, fm = lane >> 2;
  const int mc = a.m_cell;
  const int nct = a.n_col_tiles;
  const int n_mtiles = (mc + 7) / 8;
  const int mtp = a.mw / 8;            // 8-row output tiles per matrix block (= per tile of this kernel)
  const int np = a.n_parts;
  const int mt0 = warp_m * MT;
  const double alpha = a.alpha, beta = a.beta;

  if (tid == 0) {
    for (int s = 0; s < kP2Stages; ++s) { mbar_init(&full[s], 1); mbar_init(&empty[s], kP2Threads / 32); }
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    ticket_s[0] = (long long)(atomicAdd(pd.counter, 1ull) - pd.ticket_base);
  }
  __syncthreads();

  uint32_t q0 = 0;   // running panel count: ring slot = q % stages, phase = (q / stages) & 1
  for (int iter = 0;; ++iter) {
    const long long ticket = ticket_s[iter & 1];
    if (ticket >= pd.n_tiles) break;
    const int pos = (int)(ticket / (np * nct)), part = (int)((ticket / nct) % np), jt = (int)(ticket % nct);
    const int cell = pd.pos_cell[pos];
    const int row0 = part * a.mw;                                        // first output node of this tile
    const int nmt = max(0, min(MT, min(mtp, n_mtiles - part * mtp) - mt0));
    const int col0 = jt * kP2TileN;
    const int ncols = min(kP2TileN, a.B - col0);             // even (whole column pairs); the TMA zero-fills beyond B
    const int kt = a.ktot[cell];
    const int32_t* gi = a.gidx + a.idx_off[cell];
    const S* M = a.mat + a.mat_off[cell] + (int64_t)part * kt * lda;
    if (tid == 0) ticket_s[(iter + 1) & 1] = (long long)(atomicAdd(pd.counter, 1ull) - pd.ticket_base);
    const bool use_t = (beta != 0.0) && !a.atomic;   // the -beta Y_{k-2} term seeds the accumulators (below)
    for (int k = tid; k < kt; k += kP2Threads) {
      const int idx = gi[k];
      idx_s[k] = idx;
    }
    __syncthreads();

    const int npanel = kt / kP2PanelK;
    // Producer duty rotates over the 8 warps (panel j is issued by lane 0 of warp j % 8, kP2Ahead iterations ahead):
    // wait for the ring slot, then one expect_tx, one bulk copy (matrix panel) and two TMA row gathers (X or P rows).
    auto produce = [&](int pj) {
      if (lane != 0) return;
      const uint32_t q = q0 + (uint32_t)pj;
      const int s = (int)(q % kP2Stages);
      mbar_wait(&empty[s], ((q / kP2Stages) & 1u) ^ 1u);
      S* As = stage0 + s * stage_elems;
      S* Xs = As + a_panel_elems;
      const uint32_t a_bytes = (uint32_t)a_panel_elems * (uint32_t)sizeof(S);
      mbar_expect_tx(&full[s], a_bytes + (uint32_t)(kP2PanelK * kP2LdXs * sizeof(S)));
      bulk_g2s(As, M + (int64_t)pj * a_panel_elems, a_bytes, &full[s]);
      const int k0 = pj * kP2PanelK;
      const CUtensorMap* tm = (k0 < a.mpad) ? &tmX : &tmP;
      tma_gather4(Xs, tm, col0, idx_s[k0] & 0x7fffffff, idx_s[k0 + 1] & 0x7fffffff, idx_s[k0 + 2] & 0x7fffffff,
                  idx_s[k0 + 3] & 0x7fffffff, &full[s]);
      tma_gather4(Xs + 4 * kP2LdXs, tm, col0, idx_s[k0 + 4] & 0x7fffffff, idx_s[k0 + 5] & 0x7fffffff,
                  idx_s[k0 + 6] & 0x7fffffff, idx_s[k0 + 7] & 0x7fffffff, &full[s]);
    };
    if (warp < kP2Ahead && warp < npanel) produce(warp);

    const int nt0 = warp_n * 2;
    const int nnt = max(0, min(2, (ncols + 7) / 8 - nt0));
    const bool ok0 = nt0 * 8 + fk * 2 < ncols, ok1 = nt0 * 8 + 8 + fk * 2 < ncols;   // this lane's two column pairs
    const bool active = (nnt > 0 && nmt > 0);
    // Recurrence term -beta Y_{k-2} (Eq. 37): the accumulators of the first-contribution nodes START at
    // (-beta/alpha) Y_{k-2} (the target block still holds Y_{k-2}); the loads land straight in the accumulator
    // registers while the first panels are in flight, and the epilogue has no loads left.
    double acc[MT][2][2];
#pragma unroll
    for (int i = 0; i < MT; ++i)
#pragma unroll
      for (int j = 0; j < 2; ++j) acc[i][j][0] = acc[i][j][1] = 0.0;
    if (use_t && active) {
      const double nb = -beta / alpha;
#pragma unroll
      for (int i = 0; i < MT; ++i) {
        const int r = row0 + (mt0 + i) * 8 + fm;
        const int idx = (i < nmt && r < mc) ? idx_s[r] : 0;
        if (idx < 0) {
          const S* tp = a.Tg + (int64_t)(idx & 0x7fffffff) * a.ldt + col0 + nt0 * 8 + fk * 2;
          if (ok0) { const double2 u = ld_cg_pair(tp); acc[i][0][0] = u.x; acc[i][0][1] = u.y; }
          if (ok1) { const double2 v = ld_cg_pair(tp + 8); acc[i][1][0] = v.x; acc[i][1][1] = v.y; }
        }
      }
#pragma unroll
      for (int i = 0; i < MT; ++i)
#pragma unroll
        for (int j = 0; j < 2; ++j) { acc[i][j][0] *= nb; acc[i][j][1] *= nb; }
    }
    for (int pi = 0; pi < npanel; ++pi) {
      const uint32_t q = q0 + (uint32_t)pi;
      const int s = (int)(q % kP2Stages);
      {
        const int pj = pi + kP2Ahead;
        if (pj < npanel && (pj & 7) == warp) produce(pj);
      }
      mbar_wait(&full[s], (q / kP2Stages) & 1u);
      if (active) {
        const S* As = stage0 + s * stage_elems;
        const S* Ap = As + fk * lda + mt0 * 8 + fm;
        const S* Xp = As + a_panel_elems + fk * kP2LdXs + nt0 * 8 + fm;
        if (nmt == MT && nnt == 2) {
#pragma unroll
          for (int ks = 0; ks < kP2PanelK / 4; ++ks) {
            const double b0 = (double)Xp[ks * 4 * kP2LdXs], b1 = (double)Xp[ks * 4 * kP2LdXs + 8];
#pragma unroll
            for (int i = 0; i < MT; ++i) {
              const double av = (double)Ap[ks * 4 * lda + i * 8];
              dmma884(acc[i][0][0], acc[i][0][1], av, b0);
              dmma884(acc[i][1][0], acc[i][1][1], av, b1);
            }
          }
        } else {
#pragma unroll
          for (int ks = 0; ks < kP2PanelK / 4; ++ks) {
            const double b0 = (double)Xp[ks * 4 * kP2LdXs], b1 = (nnt > 1) ? (double)Xp[ks * 4 * kP2LdXs + 8] : 0.0;
#pragma unroll
            for (int i = 0; i < MT; ++i) {
              if (i < nmt) {
                const double av = (double)Ap[ks * 4 * lda + i * 8];
                dmma884(acc[i][0][0], acc[i][0][1], av, b0);
                dmma884(acc[i][1][0], acc[i][1][1], av, b1);
              }
            }
          }
        }
      }
      __syncwarp();
      if (lane == 0) mbar_arrive(&empty[s]);
    }
    q0 += (uint32_t)npanel;

    // ---- epilogue: assembly + recurrence (steps 4-5).  C fragment: row = lane/4, columns 2*(lane%4) + {0,1}
    if (!a.atomic) {
      const int d0 = pd.dep_ptr[pos], nd = (pd.dep_ptr[pos + 1] - d0) * np;   // every block of every earlier neighbour
      for (int d = lane; d < nd; d += 32) {
        const uint32_t* f = pd.flags + ((int64_t)pd.dep_pos[d0 + d / np] * np + d % np) * nct + jt;
        while (ld_acquire_gpu(f) != pd.epoch) __nanosleep(64);
      }
      __syncwarp();
    }
    if (active) {
      // first contribution to a dof: plain store of alpha acc (the -beta Y_{k-2} term is already in acc); later
      // contributions: red.global.add.f64 (fire and forget); their order is fixed by the completion flags.
#pragma unroll
      for (int i = 0; i < MT; ++i) {
        const int r = row0 + (mt0 + i) * 8 + fm;
        if (i >= nmt || r >= mc) continue;
        const int idx = idx_s[r];
        S* trow = a.Tg + (int64_t)(idx & 0x7fffffff) * a.ldt + col0 + nt0 * 8 + fk * 2;
        const bool add = a.atomic || idx >= 0;
#pragma unroll
        for (int j = 0; j < 2; ++j) {
          if (!(j ? ok1 : ok0)) continue;
          const double v0 = alpha * acc[i][j][0], v1 = alpha * acc[i][j][1];
          if (add) {
            atomicAdd(trow + j * 8, (S)v0);
            atomicAdd(trow + j * 8 + 1, (S)v1);
          } else {
            st_pair(trow + j * 8, v0, v1);
          }
        }
      }
    }
    __threadfence();
    __syncthreads();   // all stores of the tile are done and fenced; idx_s / ticket slot may be reused
    if (tid == 0 && !a.atomic) st_release_gpu(pd.flags + ((int64_t)pos * np + part) * nct + jt, pd.epoch);
  }
}

// -------------------------------------------------------------------------------------------------------------
// Steps 3a-3b as a TMA row stream (default when the block is 16-byte aligned; k_proj_rows above is the fallback).
// CTA = (row segment of <= 128 dofs, 256-column tile); the rows are gathered by tile::gather4 (box = 256 columns)
// into a 6-stage ring of 8 rows, 96 KB in flight per CTA and two CTAs per SM, so the stream does not depend on
// per-thread loads in flight; thread t owns column t of the tile and accumulates the 8 projector coefficients of the
// group over the rows of the segment in row order (no cross-thread reduction): deterministic.  HBM-bound.
// -------------------------------------------------------------------------------------------------------------
constexpr int kPTRows = 8, kPTStages = 6, kPTAhead = kPTStages - 2;
template <typename T>
size_t pt_smem_bytes(bool cplx = false) {
  return (size_t)kPTStages * kPTRows * kPRCols * sizeof(T) + (size_t)(cplx ? 2 : 1) * kProjSegRows * kProjGroup * sizeof(T) +
         (size_t)(kProjSegRows + 8) * sizeof(int32_t) + 2 * kPTStages * sizeof(uint64_t);
}
// CPLX (k-point variant): the columns are (re, im) pairs and the coefficients complex, P = conj(C)^T X (Eq. 33 with the
// Bloch phases): the thread of a real column adds  cr x_own + ci x_partner  (even column: Re P = cr xr + ci xi;
// odd column: Im P = cr xi - ci xr).
template <typename T, bool CPLX>
__global__ void __launch_bounds__(256, 2) k_proj_rows_tma(const int32_t* __restrict__ seg_ptr, const int32_t* __restrict__ grow_dof,
                                                          const T* __restrict__ pcoef, const T* __restrict__ pcoef_im,
                                                          double* __restrict__ Pc, int B,
                                                          const __grid_constant__ CUtensorMap tmX) {
  extern __shared__ __align__(128) unsigned char smem_raw[];
  T* ring = reinterpret_cast<T*>(smem_raw);                                        // [stages][8 rows][256 columns]
  T* cs = ring + kPTStages * kPTRows * kPRCols;                                    // [128][8] (+ [128][8] imaginary parts)
  T* csi = cs + kProjSegRows * kProjGroup;
  int32_t* dofs = reinterpret_cast<int32_t*>(cs + (CPLX ? 2 : 1) * kProjSegRows * kProjGroup);     // [128 + 8]
  uint64_t* full = reinterpret_cast<uint64_t*>(dofs + kProjSegRows + 8);
  uint64_t* empty = full + kPTStages;
  const int seg = blockIdx.x;
  const int r0 = seg_ptr[seg], nr = seg_ptr[seg + 1] - r0;
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  const int col0 = blockIdx.y * kPRCols;
  for (int e = tid; e < nr * kProjGroup; e += 256) {
    cs[e] = pcoef[(int64_t)r0 * kProjGroup + e];
    if (CPLX) csi[e] = pcoef_im[(int64_t)r0 * kProjGroup + e];
  }
  for (int e = tid; e < kProjSegRows + 8; e += 256) dofs[e] = grow_dof[r0 + min(e, nr - 1)];   // tail: any valid row
  if (tid == 0) {
    for (int s = 0; s < kPTStages; ++s) { mbar_init(&full[s], 1); mbar_init(&empty[s], 8); }
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
  }
  __syncthreads();
  const int npanel = (nr + kPTRows - 1) / kPTRows;
  auto produce = [&](int pj) {
    if (lane != 0) return;
    const int s = pj % kPTStages;
    mbar_wait(&empty[s], ((pj / kPTStages) & 1) ^ 1);
    const int k0 = pj * kPTRows;
    const int rows = min(kPTRows, (nr - k0 + 3) / 4 * 4);
    mbar_expect_tx(&full[s], (uint32_t)(rows * kPRCols * sizeof(T)));
    for (int r = 0; r < rows; r += 4)
      tma_gather4(ring + (s * kPTRows + r) * kPRCols, &tmX, col0, dofs[k0 + r], dofs[k0 + r + 1], dofs[k0 + r + 2],
                  dofs[k0 + r + 3], &full[s]);
  };
  if (warp < kPTAhead && warp < npanel) produce(warp);
  double acc[kProjGroup];
#pragma unroll
  for (int i = 0; i < kProjGroup; ++i) acc[i] = 0.0;
  for (int pi = 0; pi < npanel; ++pi) {
    const int s = pi % kPTStages;
    {
      const int pj = pi + kPTAhead;
      if (pj < npanel && (pj & 7) == warp) produce(pj);
    }
    mbar_wait(&full[s], (pi / kPTStages) & 1);
    const int rows = min(kPTRows, nr - pi * kPTRows);
    const T* xs = ring + s * kPTRows * kPRCols + tid;
    const T* cp = cs + pi * kPTRows * kProjGroup;
#pragma unroll 4
    for (int r = 0; r < rows; ++r) {
      const double x = (double)xs[r * kPRCols];
#pragma unroll
      for (int i = 0; i < kProjGroup; ++i) acc[i] = fma((double)cp[r * kProjGroup + i], x, acc[i]);
      if (CPLX) {
        const double xp = (tid & 1) ? -(double)xs[r * kPRCols - 1] : (double)xs[r * kPRCols + 1];   // partner column of the pair
        const T* ci = csi + (pi * kPTRows + r) * kProjGroup;
#pragma unroll
        for (int i = 0; i < kProjGroup; ++i) acc[i] = fma((double)ci[i], xp, acc[i]);
      }
    }
    __syncwarp();
    if (lane == 0) mbar_arrive(&empty[s]);
  }
  const int col = col0 + tid;
  if (col < B) {
#pragma unroll
    for (int i = 0; i < kProjGroup; ++i) Pc[((int64_t)seg * kProjGroup + i) * B + col] = acc[i];
  }
}

// k-point variant, Alg. 4 steps 5-6 dof by dof: T[g] += alpha sum_j C~_{g,j} (D P)_j with complex
// coefficients C~ = cr + i ci and complex P (column pairs re, im):  re: cr Pr - ci Pi,  im: cr Pi + ci Pr.  One CTA =
// (segment of <= 128 rows of one projector group, 256 real columns); the segments of one launch belong to groups of one
// colour, so no two CTAs of a launch touch the same row and a plain read-modify-write is race-free and ordered.
template <typename T>
__global__ void __launch_bounds__(256) k_proj_back(const int32_t* __restrict__ segs, const int32_t* __restrict__ seg_ptr,
                                                   const int32_t* __restrict__ grow_dof, const T* __restrict__ pcoef,
                                                   const T* __restrict__ pcoef_im, const int32_t* __restrict__ seg_slot_proj,
                                                   const T* __restrict__ P, int B, T* __restrict__ Tg, int64_t ldt, double alpha) {
  __shared__ T cs[kProjSegRows * kProjGroup], csi[kProjSegRows * kProjGroup];
  __shared__ int32_t dofs[kProjSegRows];
  const int seg = segs[blockIdx.x];
  const int r0 = seg_ptr[seg], nr = seg_ptr[seg + 1] - r0;
  const int tid = threadIdx.x;
  for (int e = tid; e < nr * kProjGroup; e += 256) {
    cs[e] = pcoef[(int64_t)r0 * kProjGroup + e];
    csi[e] = pcoef_im[(int64_t)r0 * kProjGroup + e];
  }
  for (int e = tid; e < nr; e += 256) dofs[e] = grow_dof[r0 + e];
  __syncthreads();
  const int col = blockIdx.y * 256 + tid;
  if (col >= B) return;
  double pr[kProjGroup], pp[kProjGroup];
  const double sgn = (col & 1) ? 1.0 : -1.0;
#pragma unroll
  for (int i = 0; i < kProjGroup; ++i) {
    const int j = seg_slot_proj[seg * kProjGroup + i];
    pr[i] = j >= 0 ? (double)P[(int64_t)j * B + col] : 0.0;
    pp[i] = j >= 0 ? sgn * (double)P[(int64_t)j * B + (col ^ 1)] : 0.0;
  }
  for (int r = 0; r < nr; ++r) {
    double v = 0.0;
#pragma unroll
    for (int i = 0; i < kProjGroup; ++i) v = fma((double)cs[r * kProjGroup + i], pr[i], fma((double)csi[r * kProjGroup + i], pp[i], v));
    T* tp = Tg + (int64_t)dofs[r] * ldt + col;
    *tp = (T)((double)*tp + alpha * v);
  }
}

#include "apply_tf32.cuh"
#include "apply_sf.cuh"
#include "apply_sf_ws.cuh"

// Tensor map of a row-major FP64 / FP32 block [rows][ld] restricted to its first `cols` columns, box = box_cols x 1
// (tile::gather4 picks four such rows per instruction); columns beyond `cols` read as zero.
using EncodeTiledFn = CUresult (*)(CUtensorMap*, CUtensorMapDataType, cuuint32_t, void*, const cuuint64_t*, const cuuint64_t*,
                                   const cuuint32_t*, const cuuint32_t*, CUtensorMapInterleave, CUtensorMapSwizzle,
                                   CUtensorMapL2promotion, CUtensorMapFloatOOBfill);
EncodeTiledFn encode_tiled_fn() {
  static EncodeTiledFn fn = [] {
    void* p = nullptr;
    cudaDriverEntryPointQueryResult q;
    if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &p, cudaEnableDefault, &q) != cudaSuccess ||
        q != cudaDriverEntryPointSuccess)
      p = nullptr;
    return reinterpret_cast<EncodeTiledFn>(p);
  }();
  return fn;
}
bool make_row_gather_map(CUtensorMap* tm, const void* base, int64_t rows, int64_t cols, int64_t ld, int elt, int box_cols,
                         bool swizzle128 = false) {
  EncodeTiledFn enc = encode_tiled_fn();
  if (!enc || rows < 1 || cols < 1 || (ld * elt) % 16 != 0 || (uintptr_t)base % 16 != 0) return false;
  const cuuint64_t dims[2] = {(cuuint64_t)cols, (cuuint64_t)rows};
  const cuuint64_t strides[1] = {(cuuint64_t)ld * (cuuint64_t)elt};
  const cuuint32_t box[2] = {(cuuint32_t)box_cols, 1};
  const cuuint32_t estr[2] = {1, 1};
  return enc(tm, elt == 8 ? CU_TENSOR_MAP_DATA_TYPE_FLOAT64 : CU_TENSOR_MAP_DATA_TYPE_FLOAT32, 2, const_cast<void*>(base), dims, strides, box, estr,
             CU_TENSOR_MAP_INTERLEAVE_NONE, swizzle128 ? CU_TENSOR_MAP_SWIZZLE_128B : CU_TENSOR_MAP_SWIZZLE_NONE,
             CU_TENSOR_MAP_L2_PROMOTION_L2_256B,
             CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE) == CUDA_SUCCESS;
}



template <typename S>
size_t p2_smem_bytes(const Op* op) {
  return (size_t)p2_stages<S>() * (kP2PanelK * op->lda + kP2PanelK * kP2LdXs) * sizeof(S) +
         2 * p2_stages<S>() * sizeof(uint64_t) + 2 * sizeof(long long) + (size_t)op->max_ktot * sizeof(int32_t);
}

template <typename T>
cudaError_t launch_apply_t(Op* op, const ApplyArgs& g, cudaStream_t st) {
  const int B = (int)g.B;
  T* P = reinterpret_cast<T*>(g.P);
  const T* X = reinterpret_cast<const T*>(g.X);
  T* Tg = reinterpret_cast<T*>(g.T);
  const T* mat = reinterpret_cast<const T*>(op->mat);
  cudaEvent_t ev[3] = {nullptr, nullptr, nullptr};
  const bool profiling = op->profiling && g.phase == 0;
  if (profiling) {
    if (op->prof_used + 3 > op->prof_events.size()) {
      for (int i = 0; i < 3; ++i) {
        cudaEvent_t e;
        cudaError_t ce = cudaEventCreate(&e);
        if (ce != cudaSuccess) return ce;
        op->prof_events.push_back(e);
      }
    }
    for (int i = 0; i < 3; ++i) ev[i] = op->prof_events[op->prof_used + i];
    op->prof_used += 3;
    cudaEventRecord(ev[0], st);
  }
  // row segments of a chunk start 16-byte aligned (TMA, vector loads / stores of the fragments)
  constexpr int kPer16 = 16 / (int)sizeof(T);
  const bool aligned = B % kPer16 == 0 && g.ldx % kPer16 == 0 && g.ldt % kPer16 == 0 && ((uintptr_t)g.X % 16 == 0) &&
                       ((uintptr_t)g.T % 16 == 0) && ((uintptr_t)g.P % 16 == 0) && op->max_ktot <= kMaxKtot;
  // variant 0 (automatic) / 5: the sum-factorised kernel (apply_sf.cuh) when the operator qualifies
  CUtensorMap tmX, tmP;
  CUtensorMap tmPs;
  bool use_sf = op->sf_ok && aligned && (op->variant == 0 || op->variant == 5 || op->variant == 6) && g.sync != nullptr && g.epoch > 0 &&
                make_row_gather_map(&tmX, g.X, op->n_dofs, B, g.ldx, (int)sizeof(T), sf_tile_cols<T>(), true);
  // variants 0 and 6: the warp-specialised form (apply_sf_ws.cuh).  It never reads the target block: T = alpha (..) or, with
  // g.accumulate, T += alpha (..); a three-term update with beta != 0 goes to k_apply_sf.
  const bool use_ws = use_sf && op->variant != 5 && (g.accumulate || g.beta == 0.0) &&
                      make_row_gather_map(&tmPs, g.P, op->n_proj + 1, B, B, (int)sizeof(T), sf_tile_cols<T>(), false);
  if (g.accumulate && !use_ws) return cudaErrorNotSupported;   // the caller asks apply_accumulates() first
  if (op->kpoint && !(use_ws && sizeof(T) == 8)) return cudaErrorNotSupported;   // the k-point variant has this one kernel
  if (!use_sf && op->dense_stale) {             // a dense kernel after chfsi_update_potential refreshed only the fields
    const cudaError_t re = refresh_dense_matrices(op, st);
    if (re != cudaSuccess) return re;
  }
  if (!use_sf && g.cshift != op->cur_shift) {   // once per filter call: move the spectral shift onto the matrix diagonals
    const int64_t n = op->n_cells * op->m_cell;
    k_set_diag_shift<T><<<(unsigned)((n + 255) / 256), 256, 0, st>>>(reinterpret_cast<T*>(op->mat), op->mat_off, op->idx_off,
                                                                    op->gidx, op->ktot, op->diag0, op->m_cell, op->lda, op->mw,
                                                                    op->n_cells, g.cshift);
    const cudaError_t se = cudaGetLastError();
    if (se != cudaSuccess) return se;           // cur_shift keeps describing what the matrices actually hold
    op->cur_shift = g.cshift;
    op->launches++;
  }
  const int64_t launches_before = op->launches;
  // steps 3a-3c
  double* Pc = reinterpret_cast<double*>(g.Pc);
  if (op->n_pseg > 0 && g.phase != 2) {
    dim3 g1((unsigned)op->n_pseg, (unsigned)((B + kPRCols - 1) / kPRCols));
    CUtensorMap tmXp;
    if (op->variant != 1 && make_row_gather_map(&tmXp, g.X, op->n_dofs, B, g.ldx, (int)sizeof(T), kPRCols)) {
      if (op->kpoint)
        k_proj_rows_tma<T, true><<<g1, 256, pt_smem_bytes<T>(true), st>>>(op->seg_ptr, op->grow_dof, reinterpret_cast<const T*>(op->pcoef),
                                                                          reinterpret_cast<const T*>(op->pcoef_im), Pc, B, tmXp);
      else
        k_proj_rows_tma<T, false><<<g1, 256, pt_smem_bytes<T>(), st>>>(op->seg_ptr, op->grow_dof, reinterpret_cast<const T*>(op->pcoef),
                                                                       nullptr, Pc, B, tmXp);
    } else {
      if (op->kpoint) return cudaErrorNotSupported;
      const int vec_ok = (g.ldx % 2 == 0 && (uintptr_t)g.X % 16 == 0) ? 1 : 0;
      k_proj_rows<T><<<g1, 256, 0, st>>>(op->seg_ptr, op->grow_dof, reinterpret_cast<const T*>(op->pcoef), X, g.ldx, Pc, B, vec_ok);
    }
    op->launches++;
  }
  if (g.phase != 2) {
    dim3 g2((unsigned)(op->n_proj + 1), (unsigned)((B + 127) / 128));
    k_proj_reduce<T><<<g2, 128, 0, st>>>(Pc, op->grp_seg_ptr, op->proj_grp, op->proj_slot, op->D, op->n_proj, P, B);
    op->launches++;
  }
  if (g.phase == 1) return cudaGetLastError();
  ApplyDev<T> a;
  a.mat = mat; a.mat_off = op->mat_off; a.idx_off = op->idx_off; a.ktot = op->ktot; a.gidx = op->gidx;
  a.m_cell = op->m_cell; a.mpad = op->mpad; a.lda = op->lda; a.mw = op->mw; a.n_parts = op->n_parts;
  a.X = X; a.ldx = g.ldx; a.Tg = Tg; a.ldt = g.ldt; a.P = P; a.ldp = B; a.B = B;
  a.alpha = (T)g.alpha; a.beta = (T)g.beta;
  a.atomic = op->assembly;
  a.accumulate = g.accumulate ? 1 : 0;

  // variant 4 (and 0 when the sum-factorised kernel does not apply): persistent single-launch dense kernel;
  // variant 2: one launch per colour; variant 1: generic
  bool fast2 = false, fast = false;
  int MT = (op->mw / 8 + 3) / 4;   // 8-row tiles per warp row: 11 (p=6), 8 (p=7, 8), 7, 4, 2, 1
  // variant 0: persistent single-launch kernel, FP64 DMMA accumulation for both storage types;
  // variant 3 (FP32 storage only, opt-in): persistent kernel with 3xTF32 products on the 32-bit tensor pipe -- 1.3x
  // faster, but the FP32 tensor accumulator truncates: |dY|/|Y| ~ 2e-6 per apply, Ritz values off by up to 4e-5 Ha,
  // i.e. inside the 1e-4 block tolerance but outside the 1e-5 Ha eigenvalue tolerance of the FP32 variant
  bool fast3 = false;   // 3xTF32 kernel
  const int MT16 = ((op->m_cell + 15) / 16 + 1) / 2;
  if (sizeof(T) == 4 && aligned && B % 8 == 0 && op->variant == 3 && op->n_parts == 1 && g.sync != nullptr && g.epoch > 0)
    fast3 = (MT16 == 11 || MT16 == 7 || MT16 == 4 || MT16 == 2 || MT16 == 1) && t3_smem_bytes(op) <= 113 * 1024 &&
            make_row_gather_map(&tmX, g.X, op->n_dofs, B, g.ldx, 4, kT3TileN) &&
            make_row_gather_map(&tmP, g.P, op->n_proj + 1, B, B, 4, kT3TileN);
  if (aligned && !fast3 && !use_sf && (op->variant == 0 || op->variant >= 4) && g.sync != nullptr && g.epoch > 0)
    fast2 = (MT == 11 || MT == 8 || MT == 7 || MT == 4 || MT == 2 || MT == 1) && p2_smem_bytes<T>(op) <= 113 * 1024 &&
            make_row_gather_map(&tmX, g.X, op->n_dofs, B, g.ldx, (int)sizeof(T), kP2TileN) &&
            make_row_gather_map(&tmP, g.P, op->n_proj + 1, B, B, (int)sizeof(T), kP2TileN);
  if (sizeof(T) == 8 && aligned && B % 8 == 0 && !fast2 && !use_sf && op->variant != 1 && op->n_parts == 1) fast = (MT == 11 || MT == 4 || MT == 2 || MT == 7);
  size_t smem_fast = (size_t)kStages * (kPanelK * op->lda + kPanelK * kLdXs) * sizeof(double) + kStages * sizeof(uint64_t) +
                     (size_t)op->max_ktot * sizeof(int32_t);
  if (fast && smem_fast > 227 * 1024) fast = false;

  if (op->assembly == 1 && !g.accumulate) {
    k_prefill<T><<<148 * 8, 256, 0, st>>>(Tg, g.ldt, op->n_dofs, B, a.beta);
    op->launches++;
  }
  if (profiling) {
    cudaEventRecord(ev[1], st);
    op->prof_proj_launches += op->launches - launches_before;
  }
  const int64_t launches_mid = op->launches;
  if (use_sf) {
    a.cells = nullptr; a.n_launch_cells = (int)op->n_cells;
    a.n_col_tiles = (B + sf_tile_cols<T>() - 1) / sf_tile_cols<T>();
    PersistDev pd;
    pd.pos_cell = op->color_cells; pd.dep_ptr = op->dep_ptr; pd.dep_pos = op->dep_pos;
    pd.counter = g.sync;
    pd.flags = reinterpret_cast<uint32_t*>(g.sync) + kSyncFlagOffset;
    pd.epoch = g.epoch;
    const int64_t n_tiles = op->n_cells * a.n_col_tiles;
    const unsigned grid = (unsigned)std::min<int64_t>(n_tiles, 2 * (int64_t)op->n_sm);
    pd.n_tiles = (int)n_tiles;
    pd.ticket_base = (unsigned long long)(g.epoch - 1) * (unsigned long long)(n_tiles + grid);
    SfDev sf;
    sf.coef = op->sf_coef; sf.sloc = op->sf_sloc; sf.crows = op->crows; sf.cell_proj_ptr = op->cell_proj_ptr;
    sf.cshift = g.cshift; sf.zero = 0;
    if (use_ws) {
      const unsigned gws = (unsigned)std::min<int64_t>(n_tiles, (int64_t)op->n_sm);
      pd.ticket_base = (unsigned long long)(g.epoch - 1) * (unsigned long long)(n_tiles + gws);
      if (op->kpoint) {
        if constexpr (sizeof(T) == 8) {
          switch (op->p) {
            case 1: k_apply_sf_ws<1, T, true><<<gws, kWsThreads, WsSmem<1, T, true>::bytes, st>>>(a, sf, pd, tmX, tmPs); break;
            case 2: k_apply_sf_ws<2, T, true><<<gws, kWsThreads, WsSmem<2, T, true>::bytes, st>>>(a, sf, pd, tmX, tmPs); break;
            case 3: k_apply_sf_ws<3, T, true><<<gws, kWsThreads, WsSmem<3, T, true>::bytes, st>>>(a, sf, pd, tmX, tmPs); break;
            case 4: k_apply_sf_ws<4, T, true><<<gws, kWsThreads, WsSmem<4, T, true>::bytes, st>>>(a, sf, pd, tmX, tmPs); break;
            case 5: k_apply_sf_ws<5, T, true><<<gws, kWsThreads, WsSmem<5, T, true>::bytes, st>>>(a, sf, pd, tmX, tmPs); break;
            case 6: k_apply_sf_ws<6, T, true><<<gws, kWsThreads, WsSmem<6, T, true>::bytes, st>>>(a, sf, pd, tmX, tmPs); break;
          }
        }
      } else
      switch (op->p) {
        case 1: k_apply_sf_ws<1, T, false><<<gws, kWsThreads, WsSmem<1, T>::bytes, st>>>(a, sf, pd, tmX, tmPs); break;
        case 2: k_apply_sf_ws<2, T, false><<<gws, kWsThreads, WsSmem<2, T>::bytes, st>>>(a, sf, pd, tmX, tmPs); break;
        case 3: k_apply_sf_ws<3, T, false><<<gws, kWsThreads, WsSmem<3, T>::bytes, st>>>(a, sf, pd, tmX, tmPs); break;
        case 4: k_apply_sf_ws<4, T, false><<<gws, kWsThreads, WsSmem<4, T>::bytes, st>>>(a, sf, pd, tmX, tmPs); break;
        case 5: k_apply_sf_ws<5, T, false><<<gws, kWsThreads, WsSmem<5, T>::bytes, st>>>(a, sf, pd, tmX, tmPs); break;
        case 6: k_apply_sf_ws<6, T, false><<<gws, kWsThreads, WsSmem<6, T>::bytes, st>>>(a, sf, pd, tmX, tmPs); break;
      }
      if (op->kpoint && op->n_pseg > 0) {
        for (size_t c = 0; c + 1 < op->back_color_ptr.size(); ++c) {
          const int n_seg_c = op->back_color_ptr[c + 1] - op->back_color_ptr[c];
          if (n_seg_c == 0) continue;
          dim3 gb((unsigned)n_seg_c, (unsigned)((B + 255) / 256));
          k_proj_back<T><<<gb, 256, 0, st>>>(op->back_segs + op->back_color_ptr[c], op->seg_ptr, op->grow_dof,
                                             reinterpret_cast<const T*>(op->pcoef), reinterpret_cast<const T*>(op->pcoef_im),
                                             op->seg_slot_proj, P, B, Tg, g.ldt, g.alpha);
          op->launches++;
        }
      }
    } else
    switch (op->p) {
      case 1: k_apply_sf<1, T><<<grid, kSfThreads, sf_smem_bytes<1, T>(op), st>>>(a, sf, pd, tmX); break;
      case 2: k_apply_sf<2, T><<<grid, kSfThreads, sf_smem_bytes<2, T>(op), st>>>(a, sf, pd, tmX); break;
      case 3: k_apply_sf<3, T><<<grid, kSfThreads, sf_smem_bytes<3, T>(op), st>>>(a, sf, pd, tmX); break;
      case 4: k_apply_sf<4, T><<<grid, kSfThreads, sf_smem_bytes<4, T>(op), st>>>(a, sf, pd, tmX); break;
      case 5: k_apply_sf<5, T><<<grid, kSfThreads, sf_smem_bytes<5, T>(op), st>>>(a, sf, pd, tmX); break;
      case 6: k_apply_sf<6, T><<<grid, kSfThreads, sf_smem_bytes<6, T>(op), st>>>(a, sf, pd, tmX); break;
    }
    op->launches++;
  }
  if (fast3) {
    if constexpr (sizeof(T) == 4) {
      a.cells = nullptr; a.n_launch_cells = (int)op->n_cells;
      a.n_col_tiles = (B + kT3TileN - 1) / kT3TileN;
      PersistDev pd;
      pd.pos_cell = op->color_cells; pd.dep_ptr = op->dep_ptr; pd.dep_pos = op->dep_pos;
      pd.counter = g.sync;
      pd.flags = reinterpret_cast<uint32_t*>(g.sync) + kSyncFlagOffset;
      pd.epoch = g.epoch;
      const int64_t n_tiles = op->n_cells * a.n_col_tiles;
      const unsigned grid = (unsigned)std::min<int64_t>(n_tiles, 2 * (int64_t)op->n_sm);
      pd.n_tiles = (int)n_tiles;
      pd.ticket_base = (unsigned long long)(g.epoch - 1) * (unsigned long long)(n_tiles + grid);
      const size_t sm = t3_smem_bytes(op);
      switch (MT16) {
        case 11: k_apply_tf32_p<11><<<grid, kP2Threads, sm, st>>>(a, pd, tmX, tmP); break;
        case 7: k_apply_tf32_p<7><<<grid, kP2Threads, sm, st>>>(a, pd, tmX, tmP); break;
        case 4: k_apply_tf32_p<4><<<grid, kP2Threads, sm, st>>>(a, pd, tmX, tmP); break;
        case 2: k_apply_tf32_p<2><<<grid, kP2Threads, sm, st>>>(a, pd, tmX, tmP); break;
        case 1: k_apply_tf32_p<1><<<grid, kP2Threads, sm, st>>>(a, pd, tmX, tmP); break;
      }
      op->launches++;
    }
  }
  if (fast2) {
    {
      a.cells = nullptr; a.n_launch_cells = (int)op->n_cells;
      a.n_col_tiles = (B + kP2TileN - 1) / kP2TileN;
      PersistDev pd;
      pd.pos_cell = op->color_cells; pd.dep_ptr = op->dep_ptr; pd.dep_pos = op->dep_pos;
      pd.counter = g.sync;
      pd.flags = reinterpret_cast<uint32_t*>(g.sync) + kSyncFlagOffset;
      pd.epoch = g.epoch;
      const int64_t n_tiles = op->n_cells * op->n_parts * a.n_col_tiles;
      unsigned grid = (unsigned)std::min<int64_t>(n_tiles, 2 * (int64_t)op->n_sm);
      pd.n_tiles = (int)n_tiles;
      pd.ticket_base = (unsigned long long)(g.epoch - 1) * (unsigned long long)(n_tiles + grid);
      const size_t sm = p2_smem_bytes<T>(op);
      switch (MT) {
        case 11: k_apply_dmma_p<11, T><<<grid, kP2Threads, sm, st>>>(a, pd, tmX, tmP); break;
        case 8: k_apply_dmma_p<8, T><<<grid, kP2Threads, sm, st>>>(a, pd, tmX, tmP); break;
        case 7: k_apply_dmma_p<7, T><<<grid, kP2Threads, sm, st>>>(a, pd, tmX, tmP); break;
        case 4: k_apply_dmma_p<4, T><<<grid, kP2Threads, sm, st>>>(a, pd, tmX, tmP); break;
        case 2: k_apply_dmma_p<2, T><<<grid, kP2Threads, sm, st>>>(a, pd, tmX, tmP); break;
        case 1: k_apply_dmma_p<1, T><<<grid, kP2Threads, sm, st>>>(a, pd, tmX, tmP); break;
      }
      op->launches++;
    }
  }
  const int n_launch = (fast2 || fast3 || use_sf) ? 0 : (op->assembly == 1 ? 1 : op->n_colors);
  for (int c = 0; c < n_launch; ++c) {
    if (op->assembly == 1) { a.cells = op->all_cells; a.n_launch_cells = (int)op->n_cells; }
    else { a.cells = op->color_cells + op->color_ptr[c]; a.n_launch_cells = op->color_ptr[c + 1] - op->color_ptr[c]; }
    if (a.n_launch_cells == 0) continue;
    if (fast) {
      if constexpr (sizeof(T) == 8) {
        a.n_col_tiles = (B + kTileN - 1) / kTileN;
        unsigned grid = (unsigned)a.n_launch_cells * (unsigned)a.n_col_tiles;
        ApplyDev<double> ad = *reinterpret_cast<ApplyDev<double>*>(&a);
        switch (MT) {
          case 11: k_apply_dmma<11><<<grid, 512, smem_fast, st>>>(ad); break;
          case 7: k_apply_dmma<7><<<grid, 512, smem_fast, st>>>(ad); break;
          case 4: k_apply_dmma<4><<<grid, 512, smem_fast, st>>>(ad); break;
          case 2: k_apply_dmma<2><<<grid, 512, smem_fast, st>>>(ad); break;
        }
      }
    } else {
      a.n_col_tiles = (B + 31) / 32;
      unsigned grid = (unsigned)a.n_launch_cells * (unsigned)a.n_col_tiles;
      k_apply_generic<T><<<grid, 256, (size_t)op->max_ktot * 32 * sizeof(T), st>>>(a);
    }
    op->launches++;
  }
  if (profiling) {
    cudaEventRecord(ev[2], st);
    op->prof_main_launches += op->launches - launches_mid;
  }
  return cudaGetLastError();
}

}  // namespace

cudaError_t init_apply_kernels(Op* op) {
  cudaError_t e;
  if ((e = init_rr_kernels())) return e;
  size_t smem_fast = (size_t)kStages * (kPanelK * op->lda + kPanelK * kLdXs) * sizeof(double) + kStages * sizeof(uint64_t) +
                     (size_t)op->max_ktot * sizeof(int32_t);
  if (smem_fast <= 227 * 1024) {
    if ((e = cudaFuncSetAttribute(k_apply_dmma<11>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem_fast))) return e;
    if ((e = cudaFuncSetAttribute(k_apply_dmma<7>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem_fast))) return e;
    if ((e = cudaFuncSetAttribute(k_apply_dmma<4>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem_fast))) return e;
    if ((e = cudaFuncSetAttribute(k_apply_dmma<2>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem_fast))) return e;
  }
  if (op->precision == 64) {
    const size_t smem_p2 = p2_smem_bytes<double>(op);
    if (smem_p2 <= 113 * 1024) {
      if ((e = cudaFuncSetAttribute(k_apply_dmma_p<11, double>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem_p2))) return e;
      if ((e = cudaFuncSetAttribute(k_apply_dmma_p<8, double>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem_p2))) return e;
      if ((e = cudaFuncSetAttribute(k_apply_dmma_p<7, double>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem_p2))) return e;
      if ((e = cudaFuncSetAttribute(k_apply_dmma_p<4, double>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem_p2))) return e;
      if ((e = cudaFuncSetAttribute(k_apply_dmma_p<2, double>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem_p2))) return e;
      if ((e = cudaFuncSetAttribute(k_apply_dmma_p<1, double>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem_p2))) return e;
    }
  } else {
    const size_t smem_p2 = p2_smem_bytes<float>(op);
    if (smem_p2 <= 113 * 1024) {
      if ((e = cudaFuncSetAttribute(k_apply_dmma_p<11, float>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem_p2))) return e;
      if ((e = cudaFuncSetAttribute(k_apply_dmma_p<8, float>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem_p2))) return e;
      if ((e = cudaFuncSetAttribute(k_apply_dmma_p<7, float>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem_p2))) return e;
      if ((e = cudaFuncSetAttribute(k_apply_dmma_p<4, float>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem_p2))) return e;
      if ((e = cudaFuncSetAttribute(k_apply_dmma_p<2, float>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem_p2))) return e;
      if ((e = cudaFuncSetAttribute(k_apply_dmma_p<1, float>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem_p2))) return e;
    }
    const size_t smem_t3 = t3_smem_bytes(op);
    if (smem_t3 <= 113 * 1024) {
      if ((e = cudaFuncSetAttribute(k_apply_tf32_p<11>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem_t3))) return e;
      if ((e = cudaFuncSetAttribute(k_apply_tf32_p<7>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem_t3))) return e;
      if ((e = cudaFuncSetAttribute(k_apply_tf32_p<4>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem_t3))) return e;
      if ((e = cudaFuncSetAttribute(k_apply_tf32_p<2>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem_t3))) return e;
      if ((e = cudaFuncSetAttribute(k_apply_tf32_p<1>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem_t3))) return e;
    }
  }
  if ((e = cudaFuncSetAttribute(k_proj_rows_tma<double, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)pt_smem_bytes<double>()))) return e;
  if ((e = cudaFuncSetAttribute(k_proj_rows_tma<float, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)pt_smem_bytes<float>()))) return e;
  if ((e = cudaFuncSetAttribute(k_proj_rows_tma<double, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)pt_smem_bytes<double>(true)))) return e;
  size_t smem_gen = (size_t)op->max_ktot * 32 * 8;
  if (smem_gen > 227 * 1024) return cudaErrorInvalidValue;
  if ((e = cudaFuncSetAttribute(k_apply_generic<double>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem_gen))) return e;
  if ((e = cudaFuncSetAttribute(k_apply_generic<float>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem_gen))) return e;
  return cudaSuccess;
}


namespace {
__global__ void __launch_bounds__(256) k_sf_sloc(const int32_t* __restrict__ gidx, const int64_t* __restrict__ idx_off,
                                                 const double* __restrict__ mass, int m_cell, int mpad, int64_t n_cells,
                                                 double* __restrict__ sloc) {
  const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= n_cells * mpad) return;
  const int64_t c = i / mpad;
  const int l = (int)(i - c * mpad);
  sloc[i] = l < m_cell ? 1.0 / sqrt(mass[gidx[idx_off[c] + l] & 0x7fffffff]) : 0.0;
}
template <int P>
cudaError_t sf_set_attr(Op* op) {
  cudaError_t e;
  if ((e = cudaFuncSetAttribute(k_apply_sf<P, double>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sf_smem_bytes<P, double>(op)))) return e;
  if ((e = cudaFuncSetAttribute(k_apply_sf_ws<P, double, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, WsSmem<P, double>::bytes))) return e;
  if ((e = cudaFuncSetAttribute(k_apply_sf_ws<P, float, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, WsSmem<P, float>::bytes))) return e;
  if ((e = cudaFuncSetAttribute(k_apply_sf_ws<P, double, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, WsSmem<P, double, true>::bytes))) return e;
  return cudaFuncSetAttribute(k_apply_sf<P, float>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sf_smem_bytes<P, float>(op));
}
}  // namespace

cudaError_t init_sf_variant(Op* op, const Tables1D& tab, cudaStream_t st) {
  op->sf_ok = false;
  if (op->p > 6 || (!op->kpoint && op->max_ktot - op->mpad > kSfMaxProj)) return cudaSuccess;   // (k-point variant: no projector data in the kernel)
  const int n1 = tab.n1, nq1 = tab.nq1;
  // Phi[q][i] = l_i(x_q): the Lagrange (GLL) basis at the Gauss points; Dh[q'][q] = derivative of the Lagrange polynomial
  // through the GAUSS points at Gauss point q' (barycentric form, long double), both zero-padded to 8 x 8
  double phi[64], dh[64];
  for (int i = 0; i < 64; ++i) phi[i] = dh[i] = 0.0;
  for (int q = 0; q < nq1; ++q)
    for (int i = 0; i < n1; ++i) phi[q * 8 + i] = tab.phi[(size_t)q * n1 + i];
  long double lam[8];
  for (int j = 0; j < nq1; ++j) {
    lam[j] = 1.0L;
    for (int k = 0; k < nq1; ++k)
      if (k != j) lam[j] /= ((long double)tab.gq_x[j] - (long double)tab.gq_x[k]);
  }
  for (int i = 0; i < nq1; ++i) {
    long double diag = 0.0L;
    for (int j = 0; j < nq1; ++j) {
      if (j == i) continue;
      const long double v = (lam[j] / lam[i]) / ((long double)tab.gq_x[i] - (long double)tab.gq_x[j]);
      dh[i * 8 + j] = (double)v;
      diag -= v;
    }
    dh[i * 8 + i] = (double)diag;
  }
  cudaError_t e;
  if ((e = cudaMemcpyToSymbolAsync(c_sf_phi, phi, sizeof(phi), (size_t)op->p * sizeof(phi), cudaMemcpyHostToDevice, st))) return e;
  if ((e = cudaMemcpyToSymbolAsync(c_sf_dhat, dh, sizeof(dh), (size_t)op->p * sizeof(dh), cudaMemcpyHostToDevice, st))) return e;
  if ((e = cudaStreamSynchronize(st))) return e;       // phi / dh live on this stack frame
  const int64_t n = op->n_cells * op->mpad;
  if ((e = cudaMalloc((void**)&op->sf_sloc, (size_t)n * sizeof(double)))) return e;
  k_sf_sloc<<<(unsigned)((n + 255) / 256), 256, 0, st>>>(op->gidx, op->idx_off, op->mass, op->m_cell, op->mpad, op->n_cells, op->sf_sloc);
  if ((e = cudaGetLastError())) return e;
  switch (op->p) {
    case 1: e = sf_set_attr<1>(op); break;
    case 2: e = sf_set_attr<2>(op); break;
    case 3: e = sf_set_attr<3>(op); break;
    case 4: e = sf_set_attr<4>(op); break;
    case 5: e = sf_set_attr<5>(op); break;
    case 6: e = sf_set_attr<6>(op); break;
  }
  if (e != cudaSuccess) return e;
  op->sf_ok = true;
  return cudaSuccess;
}

namespace {
// Dof-centric projector coefficients coef[row][slot] = sum over the cells of the row's dof of the projector rows that the
// cell matrices hold right now (Alg. 4's assembly over cells applied to C once, in the caller's CSR order: deterministic).
// *d_rows_out (optional) receives the compact device copy [nnz_cp][mpad] of those rows; the caller owns it.
cudaError_t projector_coefficients(Op* op, const HostPlan& plan, const chfsi_mesh& mesh, cudaStream_t st,
                                   std::vector<double>* coef_out, double** d_rows_out) {
  cudaError_t e;
  const int mc = op->m_cell;
  // 1. compact FP64 copy of the projector rows of the cell matrices ([nnz_cp][mpad], zero-padded), on the host
  std::vector<int32_t> row_cell((size_t)op->nnz_cp);
  for (int64_t c = 0; c < op->n_cells; ++c)
    for (int64_t r = plan.cell_proj_ptr[c]; r < plan.cell_proj_ptr[c + 1]; ++r) row_cell[r] = (int32_t)c;
  int32_t* d_row_cell = nullptr; double* d_rows = nullptr;
  if ((e = cudaMalloc((void**)&d_row_cell, row_cell.size() * sizeof(int32_t)))) return e;
  const int mpad = op->mpad;
  if ((e = cudaMalloc((void**)&d_rows, (size_t)op->nnz_cp * mpad * sizeof(double)))) { cudaFree(d_row_cell); return e; }
  std::vector<double> rows((size_t)op->nnz_cp * mpad);
  e = cudaMemcpyAsync(d_row_cell, row_cell.data(), row_cell.size() * sizeof(int32_t), cudaMemcpyHostToDevice, st);
  if (e == cudaSuccess) {
    if (op->precision == 64)
      k_extract_proj_rows<double><<<(unsigned)op->nnz_cp, 128, 0, st>>>(reinterpret_cast<const double*>(op->mat), op->mat_off,
                                                                       op->cell_proj_ptr, d_row_cell, op->ktot, mc, op->mpad, op->lda, op->mw, d_rows);
    else
      k_extract_proj_rows<float><<<(unsigned)op->nnz_cp, 128, 0, st>>>(reinterpret_cast<const float*>(op->mat), op->mat_off,
                                                                      op->cell_proj_ptr, d_row_cell, op->ktot, mc, op->mpad, op->lda, op->mw, d_rows);
    e = cudaGetLastError();
  }
  if (e == cudaSuccess) e = cudaMemcpyAsync(rows.data(), d_rows, rows.size() * sizeof(double), cudaMemcpyDeviceToHost, st);
  if (e == cudaSuccess) e = cudaStreamSynchronize(st);
  cudaFree(d_row_cell);
  if (e != cudaSuccess || !d_rows_out) cudaFree(d_rows);
  if (e != cudaSuccess) return e;
  if (d_rows_out) *d_rows_out = d_rows;
  // 2. assembly over the cells of each projector, in the caller's CSR order (deterministic)
  std::vector<double>& coef = *coef_out;
  coef.assign((size_t)op->n_prow * kProjGroup, 0.0);
  std::vector<int32_t> loc((size_t)op->n_dofs, -1);
  for (int grp = 0; grp < plan.n_groups; ++grp) {
    for (int32_t r = plan.grp_row_ptr[grp]; r < plan.grp_row_ptr[grp + 1]; ++r) loc[plan.grow_dof[r]] = r;
    for (int i = 0; i < kProjGroup; ++i) {
      const int32_t j = plan.grp_proj[(size_t)grp * kProjGroup + i];
      if (j < 0) continue;
      for (int64_t k = plan.proj_ptr[j]; k < plan.proj_ptr[j + 1]; ++k) {
        const int64_t pr = plan.proj_pcrow[k];
        const int64_t c = row_cell[pr];
        for (int l = 0; l < mc; ++l) coef[(size_t)loc[mesh.cell_dofs[c * mc + l]] * kProjGroup + i] += rows[(size_t)pr * mpad + l];
      }
    }
  }
  return cudaSuccess;
}
// upload in the operator's storage type
cudaError_t upload_coefficients(Op* op, const std::vector<double>& coef, void** dst, cudaStream_t st) {
  const size_t elt = op->precision == 64 ? 8 : 4;
  cudaError_t e;
  if ((e = cudaMalloc(dst, coef.size() * elt))) return e;
  if (op->precision == 64) {
    e = cudaMemcpyAsync(*dst, coef.data(), coef.size() * sizeof(double), cudaMemcpyHostToDevice, st);
    if (e == cudaSuccess) e = cudaStreamSynchronize(st);
  } else {
    std::vector<float> cf(coef.begin(), coef.end());
    e = cudaMemcpyAsync(*dst, cf.data(), cf.size() * sizeof(float), cudaMemcpyHostToDevice, st);
    if (e == cudaSuccess) e = cudaStreamSynchronize(st);
  }
  return e;
}
}  // namespace

cudaError_t assemble_projector_rows(Op* op, const HostPlan& plan, const chfsi_mesh& mesh, cudaStream_t st) {
  op->n_pseg = 0; op->n_prow = (int64_t)plan.grow_dof.size();
  if (op->n_proj == 0 || op->n_prow == 0 || op->nnz_cp == 0) return cudaSuccess;
  std::vector<double> coef;
  // the compact rows are kept: the sum-factorised kernels apply C~^c P from them (freed with the operator)
  cudaError_t e = projector_coefficients(op, plan, mesh, st, &coef, &op->crows);
  if (e != cudaSuccess) return e;
  if ((e = upload_coefficients(op, coef, &op->pcoef, st))) return e;
  op->n_pseg = (int64_t)plan.seg_ptr.size() - 1;
  return cudaSuccess;
}

cudaError_t assemble_projector_rows_imag(Op* op, const HostPlan& plan, const chfsi_mesh& mesh, cudaStream_t st) {
  if (op->n_pseg == 0) return cudaSuccess;
  std::vector<double> coef;
  cudaError_t e = projector_coefficients(op, plan, mesh, st, &coef, nullptr);
  if (e != cudaSuccess) return e;
  if ((e = upload_coefficients(op, coef, &op->pcoef_im, st))) return e;
  // projector of every (segment, slot), and the segments ordered by a colouring of the groups in which two groups that
  // share a dof differ: the back-projection adds into the target block one colour per launch, so that every dof is
  // summed in one fixed order
  const int n_seg = (int)op->n_pseg;
  std::vector<int32_t> seg_slot((size_t)n_seg * kProjGroup, -1), seg_color((size_t)n_seg, 0);
  std::vector<uint32_t> used((size_t)op->n_dofs, 0u);
  int n_colors = 0;
  for (int grp = 0; grp < plan.n_groups; ++grp) {
    uint32_t mask = 0;
    for (int32_t r = plan.grp_row_ptr[grp]; r < plan.grp_row_ptr[grp + 1]; ++r) mask |= used[plan.grow_dof[r]];
    int col = 0;
    while (col < 31 && (mask >> col & 1u)) ++col;
    for (int32_t r = plan.grp_row_ptr[grp]; r < plan.grp_row_ptr[grp + 1]; ++r) used[plan.grow_dof[r]] |= 1u << col;
    n_colors = std::max(n_colors, col + 1);
    for (int32_t sg = plan.grp_seg_ptr[grp]; sg < plan.grp_seg_ptr[grp + 1]; ++sg) {
      seg_color[sg] = col;
      for (int i = 0; i < kProjGroup; ++i) seg_slot[(size_t)sg * kProjGroup + i] = plan.grp_proj[(size_t)grp * kProjGroup + i];
    }
  }
  std::vector<int32_t> order;
  op->back_color_ptr.assign(1, 0);
  for (int col = 0; col < n_colors; ++col) {
    for (int sg = 0; sg < n_seg; ++sg)
      if (seg_color[sg] == col) order.push_back(sg);
    op->back_color_ptr.push_back((int32_t)order.size());
  }
  if ((e = cudaMalloc((void**)&op->seg_slot_proj, seg_slot.size() * sizeof(int32_t)))) return e;
  if ((e = cudaMalloc((void**)&op->back_segs, order.size() * sizeof(int32_t)))) return e;
  e = cudaMemcpyAsync(op->seg_slot_proj, seg_slot.data(), seg_slot.size() * sizeof(int32_t), cudaMemcpyHostToDevice, st);
  if (e == cudaSuccess) e = cudaMemcpyAsync(op->back_segs, order.data(), order.size() * sizeof(int32_t), cudaMemcpyHostToDevice, st);
  if (e == cudaSuccess) e = cudaStreamSynchronize(st);
  return e;
}

cudaError_t capture_diagonal(Op* op, cudaStream_t st) {
  const int64_t n = op->n_cells * op->m_cell;
  const unsigned grid = (unsigned)((n + 255) / 256);
  if (op->precision == 64)
    k_capture_diag<double><<<grid, 256, 0, st>>>(reinterpret_cast<const double*>(op->mat), op->mat_off, op->ktot, op->diag0,
                                                 op->m_cell, op->lda, op->mw, op->n_cells);
  else
    k_capture_diag<float><<<grid, 256, 0, st>>>(reinterpret_cast<const float*>(op->mat), op->mat_off, op->ktot, op->diag0,
                                                op->m_cell, op->lda, op->mw, op->n_cells);
  op->cur_shift = 0.0;
  return cudaGetLastError();
}

namespace {
template <typename T>
bool block_aligned(const Op* op, const ApplyArgs& g) {
  constexpr int kPer16 = 16 / (int)sizeof(T);
  return g.B % kPer16 == 0 && g.ldx % kPer16 == 0 && g.ldt % kPer16 == 0 && ((uintptr_t)g.X % 16 == 0) &&
         ((uintptr_t)g.T % 16 == 0) && ((uintptr_t)g.P % 16 == 0) && op->max_ktot <= kMaxKtot;
}
template <typename T>
__global__ void __launch_bounds__(256) k_scale_block(T* __restrict__ dst, int64_t ldd, const T* __restrict__ src, int64_t lds,
                                                     int64_t n_dofs, int B, double factor) {
  const int64_t n = n_dofs * B;
  for (int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (int64_t)gridDim.x * blockDim.x) {
    const int64_t g = i / B; const int col = (int)(i - g * B);
    dst[g * ldd + col] = (T)(factor * (double)src[g * lds + col]);
  }
}
}  // namespace

bool apply_accumulates(const Op* op, const ApplyArgs& g) {
  if (!(op->sf_ok && (op->variant == 0 || op->variant == 6) && g.sync != nullptr && encode_tiled_fn() != nullptr)) return false;
  return op->precision == 64 ? block_aligned<double>(op, g) : block_aligned<float>(op, g);
}

cudaError_t launch_scale_block(Op* op, void* dst, int64_t ldd, const void* src, int64_t lds, int64_t B, double factor,
                               cudaStream_t st) {
  const unsigned grid = (unsigned)(op->n_sm * 8);
  if (op->precision == 64)
    k_scale_block<double><<<grid, 256, 0, st>>>(reinterpret_cast<double*>(dst), ldd, reinterpret_cast<const double*>(src), lds,
                                                op->n_dofs, (int)B, factor);
  else
    k_scale_block<float><<<grid, 256, 0, st>>>(reinterpret_cast<float*>(dst), ldd, reinterpret_cast<const float*>(src), lds,
                                               op->n_dofs, (int)B, factor);
  op->launches++;
  return cudaGetLastError();
}

cudaError_t launch_apply(Op* op, const ApplyArgs& a, cudaStream_t stream) {
  return op->precision == 64 ? launch_apply_t<double>(op, a, stream) : launch_apply_t<float>(op, a, stream);
}

}  // namespace chfsi
