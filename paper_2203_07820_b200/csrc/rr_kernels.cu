// Rayleigh-Ritz projection matrices (Algorithm 2 step 1, RRGEP-OP): the overlap matrix
// S = Psi_f^T Psi_f and the projected Hamiltonian H^ = Psi_f^T (H~ Psi_f), both "X^T Y" products of two tall
// blocks [n_dofs][N] (vector index fastest) -- the paper's blocked X_p^T Y_p,
// here on one GPU with the FP64 tensor pipe.
//
//   C[i][j] = sum_g A[g][i] B[g][j]          A: [n_rows][lda], B: [n_rows][ldb], C: [N1][ldc], all FP64
//
// The stored layout is already "k-major" for both mma operands (row g = contraction index), so the fragments are
// read exactly as in the contraction kernel.  CTA tile = 128 (i) x 64 (j); 8 warps as 4 x 2, warp tile = 4 x 4
// tiles of mma.sync.m8n8k4.f64; the row range is split over gridDim.z CTAs whose partial tiles are summed in split
// order by k_xty_reduce: deterministic.  Rows stream through a 2-stage cp.async ring of 32-row panels.
#include <algorithm>

#include "common.h"

namespace chfsi {

namespace {

constexpr int kXtM = 128, kXtN = 64, kXtK = 32, kXtStages = 2;
constexpr int kXtLdA = kXtM + 4, kXtLdB = kXtN + 4;   // pitch mod 16 == 4: conflict-free 64-bit fragment loads

__device__ __forceinline__ void dmma884(double& c0, double& c1, double a, double b) {
  asm("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1}, {%2}, {%3}, {%0,%1};" : "+d"(c0), "+d"(c1) : "d"(a), "d"(b));
}
// 16-byte async copy; src_bytes = 0 zero-fills the destination (rows / columns outside the blocks)
__device__ __forceinline__ void cp_async16_zfill(void* dst, const void* src, int src_bytes) {
  asm volatile("cp.async.cg.shared.global [%0], [%1], 16, %2;" ::"r"((uint32_t)__cvta_generic_to_shared(dst)), "l"(src),
               "r"(src_bytes)
               : "memory");
}

__global__ void __launch_bounds__(256, 2) k_xty(const double* __restrict__ A, int64_t lda, const double* __restrict__ B,
                                                int64_t ldb, int64_t n_rows, int N1, int N2, int64_t rows_per_split,
                                                double* __restrict__ Cpart /*[gridDim.z][N1][N2]*/) {
  extern __shared__ __align__(16) double xs[];
  constexpr int stage_elems = kXtK * kXtLdA + kXtK * kXtLdB;
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  const int wm = warp >> 1, wn = warp & 1, fk = lane & 3, fm = lane >> 2;
  const int i0 = blockIdx.x * kXtM, j0 = blockIdx.y * kXtN;
  const int64_t g0 = (int64_t)blockIdx.z * rows_per_split, g1 = min(n_rows, g0 + rows_per_split);
  const int npanel = (int)((g1 - g0 + kXtK - 1) / kXtK);

  auto load_panel = [&](int pi) {
    double* As = xs + (pi % kXtStages) * stage_elems;
    double* Bs = As + kXtK * kXtLdA;
    const int64_t g = g0 + (int64_t)pi * kXtK;
#pragma unroll
    for (int t = 0; t < kXtK / 4; ++t) {               // A panel: kXtK rows x 64 chunks of 16 B
      const int e = tid + t * 256, r = e >> 6, c = (e & 63) * 2;
      const bool ok = (g + r < g1) && (i0 + c < N1);
      cp_async16_zfill(As + r * kXtLdA + c, ok ? A + (g + r) * lda + i0 + c : A, ok ? 16 : 0);
    }
#pragma unroll
    for (int t = 0; t < kXtK / 8; ++t) {               // B panel: kXtK rows x 32 chunks
      const int e = tid + t * 256, r = e >> 5, c = (e & 31) * 2;
      const bool ok = (g + r < g1) && (j0 + c < N2);
      cp_async16_zfill(Bs + r * kXtLdB + c, ok ? B + (g + r) * ldb + j0 + c : B, ok ? 16 : 0);
    }
  };
  for (int pi = 0; pi < kXtStages - 1; ++pi) {
    if (pi < npanel) load_panel(pi);
    asm volatile("cp.async.commit_group;" ::: "memory");
  }

  double acc[4][4][2];
#pragma unroll
  for (int i = 0; i < 4; ++i)
#pragma unroll
    for (int j = 0; j < 4; ++j) acc[i][j][0] = acc[i][j][1] = 0.0;

  for (int pi = 0; pi < npanel; ++pi) {
    asm volatile("cp.async.wait_group %0;" ::"n"(kXtStages - 2) : "memory");
    __syncthreads();                                   // panel pi has landed; everyone is done with panel pi-1
    if (pi + kXtStages - 1 < npanel) load_panel(pi + kXtStages - 1);
    asm volatile("cp.async.commit_group;" ::: "memory");
    const double* As = xs + (pi % kXtStages) * stage_elems;
    const double* Ap = As + fk * kXtLdA + wm * 32 + fm;
    const double* Bp = As + kXtK * kXtLdA + fk * kXtLdB + wn * 32 + fm;
#pragma unroll
    for (int ks = 0; ks < kXtK / 4; ++ks) {
      double b[4];
#pragma unroll
      for (int j = 0; j < 4; ++j) b[j] = Bp[ks * 4 * kXtLdB + j * 8];
#pragma unroll
      for (int i = 0; i < 4; ++i) {
        const double av = Ap[ks * 4 * kXtLdA + i * 8];
#pragma unroll
        for (int j = 0; j < 4; ++j) dmma884(acc[i][j][0], acc[i][j][1], av, b[j]);
      }
    }
  }
  // partial tile of this row split; C fragment: row = lane/4, columns 2*(lane%4) + {0,1}
  double* Cp = Cpart + (int64_t)blockIdx.z * N1 * N2;
#pragma unroll
  for (int i = 0; i < 4; ++i) {
    const int r = i0 + wm * 32 + i * 8 + fm;
    if (r >= N1) continue;
#pragma unroll
    for (int j = 0; j < 4; ++j) {
      const int c = j0 + wn * 32 + j * 8 + fk * 2;
      if (c < N2) Cp[(int64_t)r * N2 + c] = acc[i][j][0];
      if (c + 1 < N2) Cp[(int64_t)r * N2 + c + 1] = acc[i][j][1];
    }
  }
}

// C[i][j] = sum over the row splits, in split order
__global__ void __launch_bounds__(256) k_xty_reduce(const double* __restrict__ Cpart, int n_split, int N1, int N2,
                                                    double* __restrict__ C, int64_t ldc) {
  const int64_t e = (int64_t)blockIdx.x * 256 + threadIdx.x;
  if (e >= (int64_t)N1 * N2) return;
  double s = 0.0;
  for (int k = 0; k < n_split; ++k) s += Cpart[(int64_t)k * N1 * N2 + e];
  C[(e / N2) * ldc + (e % N2)] = s;
}

// ---------------------------------------------------------------------------------------------------------------
// Subspace transformation (Algorithm 2 step 3, RRGEP-ST; the paper's blocked "X_p Z" products,
// PAPER.md:560):   Out[g][j] = sum_i Y[g][i] Z[i][j]      Y: [n_rows][ldy] (N columns), Z: [N][ldz] (N2 columns)
// Rows are independent, so there is no reduction across CTAs: CTA tile = 128 rows x 64 columns, K = N streamed in
// 32-column panels of Y / 32-row panels of Z through a 2-stage cp.async ring; 8 warps as 4 x 2, 4 x 4 DMMA tiles each.
// ---------------------------------------------------------------------------------------------------------------
constexpr int kXzM = 128, kXzN = 64, kXzK = 32;
constexpr int kXzLdA = kXzK + 4, kXzLdB = kXzN + 4;   // 36, 68: pitch mod 16 == 4

__global__ void __launch_bounds__(256, 2) k_xz(const double* __restrict__ Y, int64_t ldy, const double* __restrict__ Z,
                                               int64_t ldz, int64_t n_rows, int N, int N2, double* __restrict__ Out,
                                               int64_t ldo) {
  extern __shared__ __align__(16) double xs[];
  constexpr int stage_elems = kXzM * kXzLdA + kXzK * kXzLdB;
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  const int wm = warp >> 1, wn = warp & 1, fk = lane & 3, fm = lane >> 2;
  const int j0 = blockIdx.x * kXzN;
  const int64_t g0 = (int64_t)blockIdx.y * kXzM;
  const int npanel = (N + kXzK - 1) / kXzK;

  auto load_panel = [&](int pi) {
    double* As = xs + (pi & 1) * stage_elems;
    double* Bs = As + kXzM * kXzLdA;
    const int k0 = pi * kXzK;
#pragma unroll
    for (int t = 0; t < 8; ++t) {                      // Y tile: 128 rows x 16 chunks of 16 B
      const int e = tid + t * 256, r = e >> 4, c = (e & 15) * 2;
      const bool ok = (g0 + r < n_rows) && (k0 + c < N);
      cp_async16_zfill(As + r * kXzLdA + c, ok ? Y + (g0 + r) * ldy + k0 + c : Y, ok ? 16 : 0);
    }
#pragma unroll
    for (int t = 0; t < 4; ++t) {                      // Z panel: 32 rows x 32 chunks
      const int e = tid + t * 256, r = e >> 5, c = (e & 31) * 2;
      const bool ok = (k0 + r < N) && (j0 + c < N2);
      cp_async16_zfill(Bs + r * kXzLdB + c, ok ? Z + (int64_t)(k0 + r) * ldz + j0 + c : Z, ok ? 16 : 0);
    }
  };
  load_panel(0);
  asm volatile("cp.async.commit_group;" ::: "memory");

  double acc[4][4][2];
#pragma unroll
  for (int i = 0; i < 4; ++i)
#pragma unroll
    for (int j = 0; j < 4; ++j) acc[i][j][0] = acc[i][j][1] = 0.0;

  for (int pi = 0; pi < npanel; ++pi) {
    asm volatile("cp.async.wait_group 0;" ::: "memory");
    __syncthreads();                                   // panel pi has landed; everyone is done with panel pi-1
    if (pi + 1 < npanel) load_panel(pi + 1);
    asm volatile("cp.async.commit_group;" ::: "memory");
    const double* As = xs + (pi & 1) * stage_elems;
    const double* Ap = As + (wm * 32 + fm) * kXzLdA + fk;          // A fragment: row m = fm, k = fk
    const double* Bp = As + kXzM * kXzLdA + fk * kXzLdB + wn * 32 + fm;
#pragma unroll
    for (int ks = 0; ks < kXzK / 4; ++ks) {
      double b[4];
#pragma unroll
      for (int j = 0; j < 4; ++j) b[j] = Bp[ks * 4 * kXzLdB + j * 8];
#pragma unroll
      for (int i = 0; i < 4; ++i) {
        const double av = Ap[i * 8 * kXzLdA + ks * 4];
#pragma unroll
        for (int j = 0; j < 4; ++j) dmma884(acc[i][j][0], acc[i][j][1], av, b[j]);
      }
    }
  }
#pragma unroll
  for (int i = 0; i < 4; ++i) {
    const int64_t r = g0 + wm * 32 + i * 8 + fm;
    if (r >= n_rows) continue;
#pragma unroll
    for (int j = 0; j < 4; ++j) {
      const int c = j0 + wn * 32 + j * 8 + fk * 2;
      if (c + 1 < N2) *reinterpret_cast<double2*>(Out + r * ldo + c) = make_double2(acc[i][j][0], acc[i][j][1]);
      else if (c < N2) Out[r * ldo + c] = acc[i][j][0];
    }
  }
}

constexpr size_t xz_smem_bytes() { return (size_t)2 * (kXzM * kXzLdA + kXzK * kXzLdB) * sizeof(double); }
constexpr size_t xty_smem_bytes() { return (size_t)kXtStages * (kXtK * kXtLdA + kXtK * kXtLdB) * sizeof(double); }

}  // namespace

// Shared-memory opt-in of the Rayleigh-Ritz kernels: a per-DEVICE attribute, so it is set for the current device at
// every operator creation (init_apply_kernels), not once per process.
cudaError_t init_rr_kernels() {
  cudaError_t e = cudaFuncSetAttribute(k_xz, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)xz_smem_bytes());
  if (e != cudaSuccess) return e;
  return cudaFuncSetAttribute(k_xty, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)xty_smem_bytes());
}

cudaError_t launch_xz(Op* op, const double* Y, int64_t ldy, const double* Z, int64_t ldz, int64_t n_rows, int N, int N2,
                      double* Out, int64_t ldo, cudaStream_t st) {
  const size_t smem = xz_smem_bytes();
  dim3 grid((unsigned)((N2 + kXzN - 1) / kXzN), (unsigned)((n_rows + kXzM - 1) / kXzM));
  k_xz<<<grid, 256, smem, st>>>(Y, ldy, Z, ldz, n_rows, N, N2, Out, ldo);
  op->launches++;
  return cudaGetLastError();
}

cudaError_t launch_xty(Op* op, const double* A, int64_t lda, const double* B, int64_t ldb, int64_t n_rows, int N1, int N2,
                       double* C, int64_t ldc, cudaStream_t st) {
  const int ti = (N1 + kXtM - 1) / kXtM, tj = (N2 + kXtN - 1) / kXtN;
  // Row splits: at least ~3 waves of 2 CTAs per SM and at least 512 rows per split; among the candidates the one
  // whose CTA count fills its last wave best (128 tiles x 7 splits = 3.03 waves would idle a quarter of the GPU).
  const int cap = 2 * op->n_sm, tiles = ti * tj;
  const int ns_max = (int)std::max<int64_t>(1, (n_rows + 511) / 512);
  const int ns_lo = std::min(ns_max, std::max(1, (3 * cap + tiles - 1) / tiles));
  int n_split = ns_lo;
  double best = 0.0;
  for (int ns = ns_lo; ns <= std::min(ns_max, 3 * ns_lo + 2); ++ns) {
    const int64_t ctas = (int64_t)tiles * ns;
    const double eff = (double)ctas / (double)(((ctas + cap - 1) / cap) * cap);
    if (eff > best + 1e-9) { best = eff; n_split = ns; }
  }
  int64_t rows_per_split = ((n_rows + n_split - 1) / n_split + kXtK - 1) / kXtK * kXtK;
  n_split = (int)((n_rows + rows_per_split - 1) / rows_per_split);
  const size_t need = (size_t)n_split * N1 * N2 * sizeof(double);
  if (need > op->rr_scratch_bytes) {
    cudaError_t e = cudaStreamSynchronize(st);         // the old scratch may still be in use on this stream
    if (e != cudaSuccess) return e;
    cudaFree(op->rr_scratch);
    op->rr_scratch = nullptr; op->rr_scratch_bytes = 0;
    if ((e = cudaMalloc(&op->rr_scratch, need)) != cudaSuccess) return e;
    op->rr_scratch_bytes = need;
  }
  const size_t smem = xty_smem_bytes();
  dim3 grid((unsigned)ti, (unsigned)tj, (unsigned)n_split);
  k_xty<<<grid, 256, smem, st>>>(A, lda, B, ldb, n_rows, N1, N2, rows_per_split, reinterpret_cast<double*>(op->rr_scratch));
  k_xty_reduce<<<(unsigned)(((int64_t)N1 * N2 + 255) / 256), 256, 0, st>>>(reinterpret_cast<const double*>(op->rr_scratch), n_split,
                                                                          N1, N2, C, ldc);
  op->launches += 2;
  return cudaGetLastError();
}

}  // namespace chfsi
