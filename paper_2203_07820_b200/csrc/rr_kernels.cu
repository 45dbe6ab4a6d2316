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
#include <mutex>

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
                                                int64_t ldb, int64_t n_rows, int N1, int N2, int64_t rows_per_split, int lower,
                                                double* __restrict__ Cpart /*[gridDim.z][N1][N2]*/) {
  extern __shared__ __align__(16) double xs[];
  constexpr int stage_elems = kXtK * kXtLdA + kXtK * kXtLdB;
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  const int wm = warp >> 1, wn = warp & 1, fk = lane & 3, fm = lane >> 2;
  const int i0 = blockIdx.x * kXtM, j0 = blockIdx.y * kXtN;
  if (lower && j0 > i0 + kXtM - 1) return;              // Hermitian result: tiles strictly above the diagonal are not computed
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
__global__ void __launch_bounds__(256) k_xty_reduce(const double* __restrict__ Cpart, int n_split, int N1, int N2, int lower,
                                                    double* __restrict__ C, int64_t ldc) {
  const int64_t e = (int64_t)blockIdx.x * 256 + threadIdx.x;
  if (e >= (int64_t)N1 * N2) return;
  if (lower && e % N2 > e / N2) return;                  // above the diagonal: filled by k_mirror_lower
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
// *flag |= 1 when Z [N][ld] (N2 columns) has a nonzero entry below its diagonal (row i > column j)
template <typename T>
__global__ void __launch_bounds__(256) k_lower_nonzero(const T* __restrict__ Z, int64_t ld, int N, int N2, int* __restrict__ flag) {
  const int64_t e = (int64_t)blockIdx.x * 256 + threadIdx.x;
  bool nz = false;
  if (e < (int64_t)N * N2) {
    const int i = (int)(e / N2), j = (int)(e % N2);
    nz = i > j && Z[(int64_t)i * ld + j] != T(0);
  }
  if (__syncthreads_or(nz) && threadIdx.x == 0) atomicOr(flag, 1);
}
template <typename T>
cudaError_t detect_lower_nonzero(Op* op, const T* Z, int64_t ld, int N, int N2, cudaStream_t st) {
  if (!op->rr_flag) {
    cudaError_t e = cudaMalloc(&op->rr_flag, sizeof(int));
    if (e != cudaSuccess) return e;
  }
  cudaError_t e = cudaMemsetAsync(op->rr_flag, 0, sizeof(int), st);
  if (e != cudaSuccess) return e;
  k_lower_nonzero<T><<<(unsigned)(((int64_t)N * N2 + 255) / 256), 256, 0, st>>>(Z, ld, N, N2, op->rr_flag);
  return cudaGetLastError();
}

constexpr int kXzM = 128, kXzN = 64, kXzK = 32;
constexpr int kXzLdA = kXzK + 4, kXzLdB = kXzN + 4;   // 36, 68: pitch mod 16 == 4

__global__ void __launch_bounds__(256, 2) k_xz(const double* __restrict__ Y, int64_t ldy, const double* __restrict__ Z,
                                               int64_t ldz, int64_t n_rows, int N, int N2, double* __restrict__ Out,
                                               int64_t ldo, const int* __restrict__ lower_nonzero) {
  extern __shared__ __align__(16) double xs[];
  constexpr int stage_elems = kXzM * kXzLdA + kXzK * kXzLdB;
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  const int wm = warp >> 1, wn = warp & 1, fk = lane & 3, fm = lane >> 2;
  const int j0 = blockIdx.x * kXzN;
  const int64_t g0 = (int64_t)blockIdx.y * kXzM;
  // upper-triangular Z (Z = L^-T of step 3b): rows i > j of column j are zero, the panels below this tile's columns are skipped
  const int Keff = (*lower_nonzero == 0) ? min(N, j0 + kXzN) : N;
  const int npanel = (Keff + kXzK - 1) / kXzK;

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
  if ((e = cudaFuncSetAttribute(k_xty, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)xty_smem_bytes()))) return e;
  if ((e = resolve_xty_static())) return e;              // device address of the static scratch of the allocation-free S
  return init_rr_mixed_kernels();
}

cudaError_t launch_xz(Op* op, const double* Y, int64_t ldy, const double* Z, int64_t ldz, int64_t n_rows, int N, int N2,
                      double* Out, int64_t ldo, cudaStream_t st) {
  const size_t smem = xz_smem_bytes();
  dim3 grid((unsigned)((N2 + kXzN - 1) / kXzN), (unsigned)((n_rows + kXzM - 1) / kXzM));
  cudaError_t e = detect_lower_nonzero(op, Z, ldz, N, N2, st);
  if (e != cudaSuccess) return e;
  k_xz<<<grid, 256, smem, st>>>(Y, ldy, Z, ldz, n_rows, N, N2, Out, ldo, op->rr_flag);
  op->launches += 2;
  return cudaGetLastError();
}

// Tiles of a TM x TN tiling of an N1 x N2 result that a kernel computes when only the lower triangle is wanted
int lower_tiles(int N1, int N2, int TM, int TN, int lower) {
  int n = 0;
  for (int i0 = 0; i0 < N1; i0 += TM)
    for (int j0 = 0; j0 < N2; j0 += TN) n += (lower && j0 > i0 + TM - 1) ? 0 : 1;
  return std::max(n, 1);
}

__global__ void __launch_bounds__(256) k_mirror_lower(double* __restrict__ C, int N, int64_t ldc) {
  const int64_t e = (int64_t)blockIdx.x * 256 + threadIdx.x;
  if (e >= (int64_t)N * N) return;
  const int r = (int)(e / N), c = (int)(e % N);
  if (c > r) C[(int64_t)r * ldc + c] = C[(int64_t)c * ldc + r];
}

// C[r][c] <- C[c][r] for c > r (only the lower triangle of the Hermitian S and H^ is computed)
cudaError_t launch_mirror_lower(Op* op, double* C, int N, int64_t ldc, cudaStream_t st) {
  k_mirror_lower<<<(unsigned)(((int64_t)N * N + 255) / 256), 256, 0, st>>>(C, N, ldc);
  op->launches++;
  return cudaGetLastError();
}

cudaError_t launch_xty(Op* op, const double* A, int64_t lda, const double* B, int64_t ldb, int64_t n_rows, int N1, int N2,
                       double* C, int64_t ldc, cudaStream_t st, int lower) {
  const int ti = (N1 + kXtM - 1) / kXtM, tj = (N2 + kXtN - 1) / kXtN;
  // Row splits: at least ~3 waves of 2 CTAs per SM and at least 512 rows per split; among the candidates the one
  // whose CTA count fills its last wave best (128 tiles x 7 splits = 3.03 waves would idle a quarter of the GPU).
  const int cap = 2 * op->n_sm, tiles = lower_tiles(N1, N2, kXtM, kXtN, lower);
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
  k_xty<<<grid, 256, smem, st>>>(A, lda, B, ldb, n_rows, N1, N2, rows_per_split, lower, reinterpret_cast<double*>(op->rr_scratch));
  k_xty_reduce<<<(unsigned)(((int64_t)N1 * N2 + 255) / 256), 256, 0, st>>>(reinterpret_cast<const double*>(op->rr_scratch), n_split,
                                                                          N1, N2, lower, C, ldc);
  op->launches += 2;
  return cudaGetLastError();
}

// ---------------------------------------------------------------------------------------------------------------
// Allocation-free S = Y^T Y (chfsi_overlap_matrix_noalloc, include/chfsi.h): k_xty's row-split partial sums go to a
// file-scope array in device memory instead of the cudaMalloc'ed op->rr_scratch, for callers that cannot allocate
// (CUDA graph capture, serving loops).  Every device that loads the library holds the kXtyStaticBytes of the array until
// the process exits.  In HOST code `g_xty_static` is only a stand-in for the symbol: its device address is looked up by
// cudaGetSymbolAddress once per device (resolve_xty_static, called with that device current at operator creation) and
// THAT pointer is what k_xty is given; device code (k_xty_reduce_static) names the array directly.
// The array is shared by every call on a device and keeps the last call's contents.  Nothing in it has to start at zero:
// every partial sum the reduction reads (splits 0 .. n_split-1, entries r >= c) is stored by the k_xty launch of the same
// call.  Two calls that overlap on the GPU (different streams, no dependency) race on it.
// ---------------------------------------------------------------------------------------------------------------
namespace {
constexpr size_t kXtyStaticDoubles = (size_t)CHFSI_NOALLOC_SPLITS * CHFSI_NOALLOC_MAX_N * CHFSI_NOALLOC_MAX_N;   // 2 Mi doubles
constexpr size_t kXtyStaticBytes = kXtyStaticDoubles * sizeof(double);                                          // 16 MiB
static __device__ __align__(256) double g_xty_static[kXtyStaticDoubles];

constexpr int kMaxDevices = 64;
double* g_xty_static_ptr[kMaxDevices] = {};         // device address of g_xty_static on device d (nullptr: not looked up yet)
std::mutex g_xty_static_mutex;

// C[r][c] (r >= c) = sum over the row splits, in split order, of the partial sums in g_xty_static
__global__ void __launch_bounds__(256) k_xty_reduce_static(int n_split, int N, double* __restrict__ C, int64_t ldc) {
  const int64_t e = (int64_t)blockIdx.x * 256 + threadIdx.x;
  if (e >= (int64_t)N * N) return;
  if (e % N > e / N) return;                            // above the diagonal: filled by k_mirror_lower
  double s = 0.0;
  for (int k = 0; k < n_split; ++k) s += g_xty_static[(int64_t)k * N * N + e];
  C[(e / N) * ldc + (e % N)] = s;
}
}  // namespace

// Once per device, with that device current (init_rr_kernels at operator creation): the device address of the array.
cudaError_t resolve_xty_static() {
  int dev = -1;
  cudaError_t e = cudaGetDevice(&dev);
  if (e != cudaSuccess) return e;
  if (dev < 0 || dev >= kMaxDevices) return cudaErrorInvalidDevice;
  std::lock_guard<std::mutex> lock(g_xty_static_mutex);
  if (g_xty_static_ptr[dev]) return cudaSuccess;
  double* ptr = nullptr;
  e = cudaGetSymbolAddress((void**)&ptr, g_xty_static);
  if (e != cudaSuccess) return e;
  if (!ptr) return cudaErrorInvalidSymbol;
  g_xty_static_ptr[dev] = ptr;
  return cudaSuccess;
}

// S[N][N] = Y^T Y, lower triangle computed and mirrored as in chfsi_overlap_matrix.  No cudaMalloc / cudaFree / event or
// stream creation: three kernel launches on `st`.  cudaErrorInvalidValue: N beyond CHFSI_NOALLOC_MAX_N;
// cudaErrorInvalidDevice: the current device is not one an operator was created on (no looked-up address).
cudaError_t launch_xty_static(Op* op, const double* Y, int64_t ldy, int64_t n_rows, int N, double* S, int64_t lds, cudaStream_t st) {
  if (N < 1 || N > CHFSI_NOALLOC_MAX_N) return cudaErrorInvalidValue;
  int dev = -1;
  cudaError_t e = cudaGetDevice(&dev);
  if (e != cudaSuccess) return e;
  double* scratch = nullptr;
  if (dev >= 0 && dev < kMaxDevices) {
    std::lock_guard<std::mutex> lock(g_xty_static_mutex);
    scratch = g_xty_static_ptr[dev];
  }
  if (!scratch) return cudaErrorInvalidDevice;         // no operator was created with this device current
  const int ti = (N + kXtM - 1) / kXtM, tj = (N + kXtN - 1) / kXtN;
  // row splits as in launch_xty, but never more than fit into the array (>= CHFSI_NOALLOC_SPLITS by construction)
  const int cap = 2 * op->n_sm, tiles = lower_tiles(N, N, kXtM, kXtN, 1);
  const int ns_fit = (int)std::min<size_t>(kXtyStaticDoubles / ((size_t)N * N), 1u << 20);
  const int ns_max = std::min(ns_fit, (int)std::max<int64_t>(1, (n_rows + 511) / 512));
  const int ns_lo = std::min(ns_max, std::max(1, (3 * cap + tiles - 1) / tiles));
  int n_split = ns_lo;
  double best = 0.0;
  for (int ns = ns_lo; ns <= std::min(ns_max, 3 * ns_lo + 2); ++ns) {
    const int64_t ctas = (int64_t)tiles * ns;
    const double eff = (double)ctas / (double)(((ctas + cap - 1) / cap) * cap);
    if (eff > best + 1e-9) { best = eff; n_split = ns; }
  }
  const int64_t rows_per_split = ((n_rows + n_split - 1) / n_split + kXtK - 1) / kXtK * kXtK;
  n_split = (int)((n_rows + rows_per_split - 1) / rows_per_split);
  if ((size_t)n_split * N * N > kXtyStaticDoubles) return cudaErrorInvalidValue;      // cannot happen: n_split <= ns_fit
  dim3 grid((unsigned)ti, (unsigned)tj, (unsigned)n_split);
  k_xty<<<grid, 256, xty_smem_bytes(), st>>>(Y, ldy, Y, ldy, n_rows, N, N, rows_per_split, 1, scratch);
  k_xty_reduce_static<<<(unsigned)(((int64_t)N * N + 255) / 256), 256, 0, st>>>(n_split, N, S, lds);
  k_mirror_lower<<<(unsigned)(((int64_t)N * N + 255) / 256), 256, 0, st>>>(S, N, lds);
  op->launches += 3;
  return cudaGetLastError();
}

}  // namespace chfsi

// =================================================================================================================
// Mixed-precision Rayleigh-Ritz products (Sec. 3.2 and 4.4.1: PAPER.md:396, 426-440, 564): the off-diagonal / occupied
// blocks of S and H^ and the off-diagonal part of Psi_f L^-T are FP32 products.  Here an FP32 product runs on the 32-bit
// tensor pipe as a 3xTF32 split (x = hi + lo, a b ~ a_lo b_hi + a_hi b_lo + a_hi b_hi: FP32-level products; single-pass
// TF32 would be narrower than the paper's FP32).  The FP32 accumulator of the tensor pipe truncates, so an accumulation
// chain is kept to ONE 32-row panel (4 k-steps from zero); panel sums are added to FP64 register totals with round to
// nearest, and the row splits of the grid are summed in FP64 in split order (deterministic).
// =================================================================================================================
namespace chfsi {
namespace {

__device__ __forceinline__ uint32_t rr_to_tf32(float x) {
  uint32_t r;
  asm("cvt.rna.tf32.f32 %0, %1;" : "=r"(r) : "f"(x));
  return r;
}
__device__ __forceinline__ void rr_split(float x, uint32_t& hi, uint32_t& lo) {
  hi = rr_to_tf32(x);
  lo = rr_to_tf32(x - __uint_as_float(hi));
}
__device__ __forceinline__ void rr_mma_tf32(float (&c)[4], const uint32_t (&a)[4], uint32_t b0, uint32_t b1) {
  asm("mma.sync.aligned.m16n8k8.row.col.f32.tf32.tf32.f32 {%0,%1,%2,%3}, {%4,%5,%6,%7}, {%8,%9}, {%0,%1,%2,%3};"
      : "+f"(c[0]), "+f"(c[1]), "+f"(c[2]), "+f"(c[3])
      : "r"(a[0]), "r"(a[1]), "r"(a[2]), "r"(a[3]), "r"(b0), "r"(b1));
}
__device__ __forceinline__ void cp_async16_zfill_f(void* dst, const void* src, int src_bytes) {
  asm volatile("cp.async.cg.shared.global [%0], [%1], 16, %2;" ::"r"((uint32_t)__cvta_generic_to_shared(dst)), "l"(src),
               "r"(src_bytes)
               : "memory");
}

// dst[r][c] (float, pitch ldd) = (float) src[r][c] (double, pitch lds), c < cols; optionally the diagonal of a square
// matrix is zeroed and returned separately (L^-T split into off-diagonal FP32 part and FP64 diagonal)
__global__ void __launch_bounds__(256) k_to_f32(const double* __restrict__ src, int64_t lds, float* __restrict__ dst, int64_t ldd,
                                               int64_t rows, int cols, int zero_diag, double* __restrict__ diag) {
  const int64_t n = rows * (int64_t)(cols / 2);
  for (int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (int64_t)gridDim.x * blockDim.x) {
    const int64_t r = i / (cols / 2);
    const int c = (int)(i % (cols / 2)) * 2;
    double2 v = *reinterpret_cast<const double2*>(src + r * lds + c);
    if (zero_diag) {
      if (r == c) { diag[r] = v.x; v.x = 0.0; }
      if (r == c + 1) { diag[r] = v.y; v.y = 0.0; }
    }
    *reinterpret_cast<float2*>(dst + r * ldd + c) = make_float2((float)v.x, (float)v.y);
  }
}

constexpr int kT32M = 128, kT32N = 64, kT32K = 32, kT32Stages = 3;
constexpr int kT32LdA = kT32M + 8, kT32LdB = kT32N + 8;       // k-major panels: pitch mod 32 == 8 -> conflict-free fragments

// Cpart[z][i][j] = sum over the rows of split z of A[g][i] B[g][j]   (A: [rows][lda] FP32, B: [rows][ldb] FP32);
// tiles that lie entirely inside a diagonal block of width `skip_block` (> 0) are skipped: those entries are FP64 products
__global__ void __launch_bounds__(256, 1) k_xty_tf32(const float* __restrict__ A, int64_t lda, const float* __restrict__ B,
                                                     int64_t ldb, int64_t n_rows, int N1, int N2, int64_t rows_per_split,
                                                     int skip_block, int row_block0, int col_block0, int lower,
                                                     double* __restrict__ Cpart) {
  extern __shared__ __align__(16) float fs[];
  constexpr int stage_elems = kT32K * kT32LdA + kT32K * kT32LdB;
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  const int wm = warp >> 1, wn = warp & 1, g = lane >> 2, t = lane & 3;
  const int i0 = blockIdx.x * kT32M, j0 = blockIdx.y * kT32N;
  double* Cp = Cpart + (int64_t)blockIdx.z * N1 * N2;
  if (lower && j0 > i0 + kT32M - 1) return;                     // strictly above the diagonal
  if (skip_block > 0) {
    const int bi0 = (row_block0 + i0) / skip_block, bi1 = (row_block0 + min(i0 + kT32M, N1) - 1) / skip_block;
    const int bj0 = (col_block0 + j0) / skip_block, bj1 = (col_block0 + min(j0 + kT32N, N2) - 1) / skip_block;
    if (bi0 == bi1 && bj0 == bj1 && bi0 == bj0) return;        // overwritten by the FP64 diagonal block
  }
  const int64_t g0 = (int64_t)blockIdx.z * rows_per_split, g1 = min(n_rows, g0 + rows_per_split);
  const int npanel = (int)((g1 - g0 + kT32K - 1) / kT32K);

  auto load_panel = [&](int pi) {
    float* As = fs + (pi % kT32Stages) * stage_elems;
    float* Bs = As + kT32K * kT32LdA;
    const int64_t gr = g0 + (int64_t)pi * kT32K;
#pragma unroll
    for (int it = 0; it < 4; ++it) {                     // A panel: 32 rows x 32 chunks of 16 B
      const int e = tid + it * 256, r = e >> 5, c = (e & 31) * 4;
      const bool ok = (gr + r < g1) && (i0 + c < N1);
      cp_async16_zfill_f(As + r * kT32LdA + c, ok ? A + (gr + r) * lda + i0 + c : A, ok ? 16 : 0);
    }
#pragma unroll
    for (int it = 0; it < 2; ++it) {                     // B panel: 32 rows x 16 chunks
      const int e = tid + it * 256, r = e >> 4, c = (e & 15) * 4;
      const bool ok = (gr + r < g1) && (j0 + c < N2);
      cp_async16_zfill_f(Bs + r * kT32LdB + c, ok ? B + (gr + r) * ldb + j0 + c : B, ok ? 16 : 0);
    }
  };
  for (int pi = 0; pi < kT32Stages - 1; ++pi) {
    if (pi < npanel) load_panel(pi);
    asm volatile("cp.async.commit_group;" ::: "memory");
  }
  double tot[2][4][4];
#pragma unroll
  for (int i = 0; i < 2; ++i)
#pragma unroll
    for (int j = 0; j < 4; ++j)
#pragma unroll
      for (int k = 0; k < 4; ++k) tot[i][j][k] = 0.0;

  for (int pi = 0; pi < npanel; ++pi) {
    asm volatile("cp.async.wait_group %0;" ::"n"(kT32Stages - 2) : "memory");
    __syncthreads();
    if (pi + kT32Stages - 1 < npanel) load_panel(pi + kT32Stages - 1);
    asm volatile("cp.async.commit_group;" ::: "memory");
    const float* As = fs + (pi % kT32Stages) * stage_elems;
    const float* Bs = As + kT32K * kT32LdA;
    float c[2][4][4];
#pragma unroll
    for (int i = 0; i < 2; ++i)
#pragma unroll
      for (int j = 0; j < 4; ++j) c[i][j][0] = c[i][j][1] = c[i][j][2] = c[i][j][3] = 0.f;
#pragma unroll
    for (int ks = 0; ks < kT32K / 8; ++ks) {
      uint32_t ah[2][4], al[2][4], bh[4][2], bl[4][2];
#pragma unroll
      for (int i = 0; i < 2; ++i) {
        const float* ap = As + (ks * 8 + t) * kT32LdA + wm * 32 + i * 16 + g;      // A fragment (m16 x k8), k-major storage
        rr_split(ap[0], ah[i][0], al[i][0]);
        rr_split(ap[8], ah[i][1], al[i][1]);
        rr_split(ap[4 * kT32LdA], ah[i][2], al[i][2]);
        rr_split(ap[4 * kT32LdA + 8], ah[i][3], al[i][3]);
      }
#pragma unroll
      for (int j = 0; j < 4; ++j) {
        const float* bp = Bs + (ks * 8 + t) * kT32LdB + wn * 32 + j * 8 + g;
        rr_split(bp[0], bh[j][0], bl[j][0]);
        rr_split(bp[4 * kT32LdB], bh[j][1], bl[j][1]);
      }
#pragma unroll
      for (int i = 0; i < 2; ++i)
#pragma unroll
        for (int j = 0; j < 4; ++j) {
          rr_mma_tf32(c[i][j], al[i], bh[j][0], bh[j][1]);
          rr_mma_tf32(c[i][j], ah[i], bl[j][0], bl[j][1]);
          rr_mma_tf32(c[i][j], ah[i], bh[j][0], bh[j][1]);
        }
    }
#pragma unroll
    for (int i = 0; i < 2; ++i)
#pragma unroll
      for (int j = 0; j < 4; ++j)
#pragma unroll
        for (int k = 0; k < 4; ++k) tot[i][j][k] += (double)c[i][j][k];
  }
  // C fragment: rows g, g + 8; columns 2t, 2t + 1
#pragma unroll
  for (int i = 0; i < 2; ++i)
#pragma unroll
    for (int h = 0; h < 2; ++h) {
      const int r = i0 + wm * 32 + i * 16 + g + 8 * h;
      if (r >= N1) continue;
#pragma unroll
      for (int j = 0; j < 4; ++j) {
        const int cc = j0 + wn * 32 + j * 8 + 2 * t;
        if (cc < N2) Cp[(int64_t)r * N2 + cc] = tot[i][j][2 * h];
        if (cc + 1 < N2) Cp[(int64_t)r * N2 + cc + 1] = tot[i][j][2 * h + 1];
      }
    }
}

// C[r][c] = sum over splits; entries of tiles skipped above are left untouched (mask by the same rule)
__global__ void __launch_bounds__(256) k_xty_reduce_masked(const double* __restrict__ Cpart, int n_split, int N1, int N2,
                                                           int skip_block, int row_block0, int col_block0, int lower,
                                                           double* __restrict__ C, int64_t ldc) {
  const int64_t e = (int64_t)blockIdx.x * 256 + threadIdx.x;
  if (e >= (int64_t)N1 * N2) return;
  const int r = (int)(e / N2), c = (int)(e % N2);
  if (lower && c > r) return;
  if (skip_block > 0) {
    const int i0 = r / kT32M * kT32M, j0 = c / kT32N * kT32N;
    const int bi0 = (row_block0 + i0) / skip_block, bi1 = (row_block0 + min(i0 + kT32M, N1) - 1) / skip_block;
    const int bj0 = (col_block0 + j0) / skip_block, bj1 = (col_block0 + min(j0 + kT32N, N2) - 1) / skip_block;
    if (bi0 == bi1 && bj0 == bj1 && bi0 == bj0) return;
  }
  double s = 0.0;
  for (int k = 0; k < n_split; ++k) s += Cpart[(int64_t)k * N1 * N2 + e];
  C[(int64_t)r * ldc + c] = s;
}

// Out[g][j] = sum_i Y32[g][i] Z32[i][j] (3xTF32, Z32 = off-diagonal part)  +  Y[g][j] zd[j] (FP64 diagonal part)
constexpr int kZ32M = 128, kZ32N = 64, kZ32K = 32;
constexpr int kZ32LdA = kZ32K + 4, kZ32LdB = kZ32N + 8;      // A row-major (m x k): pitch mod 32 == 4; B k-major: pitch mod 32 == 8
__global__ void __launch_bounds__(256, 1) k_xz_tf32(const float* __restrict__ Y32, int64_t ldy32, const float* __restrict__ Z32,
                                                    int64_t ldz32, const double* __restrict__ Y, int64_t ldy,
                                                    const double* __restrict__ zd, int64_t n_rows, int N, int N2,
                                                    double* __restrict__ Out, int64_t ldo, const int* __restrict__ lower_nonzero) {
  extern __shared__ __align__(16) float fs[];
  constexpr int stage_elems = kZ32M * kZ32LdA + kZ32K * kZ32LdB;
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  const int wm = warp >> 1, wn = warp & 1, g = lane >> 2, t = lane & 3;
  const int j0 = blockIdx.x * kZ32N;
  const int64_t g0 = (int64_t)blockIdx.y * kZ32M;
  const int Keff = (*lower_nonzero == 0) ? min(N, j0 + kZ32N) : N;      // upper-triangular Z: zero panels skipped (k_xz)
  const int npanel = (Keff + kZ32K - 1) / kZ32K;
  auto load_panel = [&](int pi) {
    float* As = fs + (pi & 1) * stage_elems;
    float* Bs = As + kZ32M * kZ32LdA;
    const int k0 = pi * kZ32K;
#pragma unroll
    for (int it = 0; it < 4; ++it) {                     // Y tile: 128 rows x 8 chunks of 16 B
      const int e = tid + it * 256, r = e >> 3, c = (e & 7) * 4;
      const bool ok = (g0 + r < n_rows) && (k0 + c < N);
      cp_async16_zfill_f(As + r * kZ32LdA + c, ok ? Y32 + (g0 + r) * ldy32 + k0 + c : Y32, ok ? 16 : 0);
    }
#pragma unroll
    for (int it = 0; it < 2; ++it) {                     // Z panel: 32 rows x 16 chunks
      const int e = tid + it * 256, r = e >> 4, c = (e & 15) * 4;
      const bool ok = (k0 + r < N) && (j0 + c < N2);
      cp_async16_zfill_f(Bs + r * kZ32LdB + c, ok ? Z32 + (int64_t)(k0 + r) * ldz32 + j0 + c : Z32, ok ? 16 : 0);
    }
  };
  load_panel(0);
  asm volatile("cp.async.commit_group;" ::: "memory");
  double tot[2][4][4];
#pragma unroll
  for (int i = 0; i < 2; ++i)
#pragma unroll
    for (int j = 0; j < 4; ++j)
#pragma unroll
      for (int k = 0; k < 4; ++k) tot[i][j][k] = 0.0;
  for (int pi = 0; pi < npanel; ++pi) {
    asm volatile("cp.async.wait_group 0;" ::: "memory");
    __syncthreads();
    if (pi + 1 < npanel) load_panel(pi + 1);
    asm volatile("cp.async.commit_group;" ::: "memory");
    const float* As = fs + (pi & 1) * stage_elems;
    const float* Bs = As + kZ32M * kZ32LdA;
    float c[2][4][4];
#pragma unroll
    for (int i = 0; i < 2; ++i)
#pragma unroll
      for (int j = 0; j < 4; ++j) c[i][j][0] = c[i][j][1] = c[i][j][2] = c[i][j][3] = 0.f;
#pragma unroll
    for (int ks = 0; ks < kZ32K / 8; ++ks) {
      uint32_t ah[2][4], al[2][4], bh[4][2], bl[4][2];
#pragma unroll
      for (int i = 0; i < 2; ++i) {
        const float* ap = As + (wm * 32 + i * 16 + g) * kZ32LdA + ks * 8 + t;      // A fragment (m16 x k8), row-major storage
        rr_split(ap[0], ah[i][0], al[i][0]);
        rr_split(ap[8 * kZ32LdA], ah[i][1], al[i][1]);
        rr_split(ap[4], ah[i][2], al[i][2]);
        rr_split(ap[8 * kZ32LdA + 4], ah[i][3], al[i][3]);
      }
#pragma unroll
      for (int j = 0; j < 4; ++j) {
        const float* bp = Bs + (ks * 8 + t) * kZ32LdB + wn * 32 + j * 8 + g;
        rr_split(bp[0], bh[j][0], bl[j][0]);
        rr_split(bp[4 * kZ32LdB], bh[j][1], bl[j][1]);
      }
#pragma unroll
      for (int i = 0; i < 2; ++i)
#pragma unroll
        for (int j = 0; j < 4; ++j) {
          rr_mma_tf32(c[i][j], al[i], bh[j][0], bh[j][1]);
          rr_mma_tf32(c[i][j], ah[i], bl[j][0], bl[j][1]);
          rr_mma_tf32(c[i][j], ah[i], bh[j][0], bh[j][1]);
        }
    }
#pragma unroll
    for (int i = 0; i < 2; ++i)
#pragma unroll
      for (int j = 0; j < 4; ++j)
#pragma unroll
        for (int k = 0; k < 4; ++k) tot[i][j][k] += (double)c[i][j][k];
  }
#pragma unroll
  for (int i = 0; i < 2; ++i)
#pragma unroll
    for (int h = 0; h < 2; ++h) {
      const int64_t r = g0 + wm * 32 + i * 16 + g + 8 * h;
      if (r >= n_rows) continue;
#pragma unroll
      for (int j = 0; j < 4; ++j) {
        const int cc = j0 + wn * 32 + j * 8 + 2 * t;
        if (cc + 1 < N2) {
          const double2 y2 = *reinterpret_cast<const double2*>(Y + r * ldy + cc);
          *reinterpret_cast<double2*>(Out + r * ldo + cc) =
              make_double2(fma(y2.x, zd[cc], tot[i][j][2 * h]), fma(y2.y, zd[cc + 1], tot[i][j][2 * h + 1]));
        } else if (cc < N2) {
          Out[r * ldo + cc] = fma(Y[r * ldy + cc], zd[cc], tot[i][j][2 * h]);
        }
      }
    }
}

constexpr size_t xty32_smem_bytes() { return (size_t)kT32Stages * (kT32K * kT32LdA + kT32K * kT32LdB) * sizeof(float); }
constexpr size_t xz32_smem_bytes() { return (size_t)2 * (kZ32M * kZ32LdA + kZ32K * kZ32LdB) * sizeof(float); }

}  // namespace

cudaError_t init_rr_mixed_kernels() {
  cudaError_t e = init_umma_kernels();
  if (e != cudaSuccess) return e;
  e = cudaFuncSetAttribute(k_xty_tf32, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)xty32_smem_bytes());
  if (e != cudaSuccess) return e;
  return cudaFuncSetAttribute(k_xz_tf32, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)xz32_smem_bytes());
}

cudaError_t launch_to_f32(Op* op, const double* src, int64_t lds, float* dst, int64_t ldd, int64_t rows, int cols, int zero_diag,
                          double* diag, cudaStream_t st) {
  const int64_t n = rows * (int64_t)(cols / 2);
  const unsigned grid = (unsigned)std::min<int64_t>((n + 255) / 256, 148 * 16);
  k_to_f32<<<grid, 256, 0, st>>>(src, lds, dst, ldd, rows, cols, zero_diag, diag);
  op->launches++;
  return cudaGetLastError();
}

cudaError_t launch_xty_tf32(Op* op, const float* A, int64_t lda, const float* B, int64_t ldb, int64_t n_rows, int N1, int N2,
                            int skip_block, int row_block0, int col_block0, double* C, int64_t ldc, cudaStream_t st, int lower) {
  const int ti = (N1 + kT32M - 1) / kT32M, tj = (N2 + kT32N - 1) / kT32N;
  const int cap = 2 * op->n_sm, tiles = lower_tiles(N1, N2, kT32M, kT32N, lower);
  const int ns_max = (int)std::max<int64_t>(1, (n_rows + 1023) / 1024);
  int n_split = std::min(ns_max, std::max(1, (3 * cap + tiles - 1) / tiles));
  int64_t rows_per_split = ((n_rows + n_split - 1) / n_split + kT32K - 1) / kT32K * kT32K;
  n_split = (int)((n_rows + rows_per_split - 1) / rows_per_split);
  if (op->rr_variant != 2)                                   // the tcgen05 kernel has its own tile shape and occupancy
    umma_xty_plan(op->n_sm, n_rows, N1, N2, skip_block, row_block0, col_block0, lower, &n_split, &rows_per_split);
  const size_t need = (size_t)n_split * N1 * N2 * sizeof(double);
  if (need > op->rr_scratch_bytes) {
    cudaError_t e = cudaStreamSynchronize(st);
    if (e != cudaSuccess) return e;
    cudaFree(op->rr_scratch);
    op->rr_scratch = nullptr; op->rr_scratch_bytes = 0;
    if ((e = cudaMalloc(&op->rr_scratch, need)) != cudaSuccess) return e;
    op->rr_scratch_bytes = need;
  }
  // rr_variant 0 / 1: the tcgen05 kernel (rr_umma.cu); 2, or no tensor maps: the mma.sync kernel below.  Same partial sums layout.
  dim3 grid((unsigned)ti, (unsigned)tj, (unsigned)n_split);
  if (op->rr_variant == 2 ||
      !launch_xty_umma(A, lda, B, ldb, n_rows, N1, N2, n_split, rows_per_split, skip_block, row_block0, col_block0, lower,
                       reinterpret_cast<double*>(op->rr_scratch), st))
    k_xty_tf32<<<grid, 256, xty32_smem_bytes(), st>>>(A, lda, B, ldb, n_rows, N1, N2, rows_per_split, skip_block, row_block0,
                                                      col_block0, lower, reinterpret_cast<double*>(op->rr_scratch));
  k_xty_reduce_masked<<<(unsigned)(((int64_t)N1 * N2 + 255) / 256), 256, 0, st>>>(
      reinterpret_cast<const double*>(op->rr_scratch), n_split, N1, N2, skip_block, row_block0, col_block0, lower, C, ldc);
  op->launches += 2;
  return cudaGetLastError();
}

cudaError_t launch_xz_tf32(Op* op, const float* Y32, int64_t ldy32, const float* Z32, int64_t ldz32, const double* Y, int64_t ldy,
                           const double* zd, int64_t n_rows, int N, int N2, double* Out, int64_t ldo, cudaStream_t st) {
  dim3 grid((unsigned)((N2 + kZ32N - 1) / kZ32N), (unsigned)((n_rows + kZ32M - 1) / kZ32M));
  cudaError_t e = detect_lower_nonzero(op, Z32, ldz32, N, N2, st);
  if (e != cudaSuccess) return e;
  if (op->rr_variant == 2 || !launch_xz_umma(Y32, ldy32, Z32, ldz32, Y, ldy, zd, n_rows, N, N2, Out, ldo, op->rr_flag, st))   // tcgen05 first
    k_xz_tf32<<<grid, 256, xz32_smem_bytes(), st>>>(Y32, ldy32, Z32, ldz32, Y, ldy, zd, n_rows, N, N2, Out, ldo, op->rr_flag);
  op->launches += 2;
  return cudaGetLastError();
}

}  // namespace chfsi
