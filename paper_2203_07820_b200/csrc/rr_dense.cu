// Dense N x N step of the Rayleigh-Ritz procedure on the device: Algorithm 2 step 2a, the Cholesky
// factorisation S = L L^T of the overlap matrix, and L^-1, which steps 2b / 3b need (H^ -> L^-1 H^ L^-T and
// Psi^o = Psi_f L^-T).  N is the number of wavefunctions (<= a few thousand on one GPU), so this is O(N^3) work on
// small matrices: blocked right-looking factorisation with 32 x 32 blocks, one launch sequence per block column
// (diagonal block -> panel solve -> trailing update), then L^-1 block row by block row.  FP64 throughout, no host
// round trip, deterministic.  (The paper runs this step on the CPUs with ScaLAPACK / ELPA.)
#include <algorithm>

#include "common.h"

namespace chfsi {
namespace {

constexpr int kNb = 32;

// L <- lower triangle of S (upper part zero)
__global__ void __launch_bounds__(256) k_copy_lower(const double* __restrict__ S, double* __restrict__ L, int N) {
  const int64_t e = (int64_t)blockIdx.x * 256 + threadIdx.x;
  if (e >= (int64_t)N * N) return;
  const int r = (int)(e / N), c = (int)(e % N);
  L[e] = (c <= r) ? S[e] : 0.0;
}

// unblocked Cholesky of the nb x nb diagonal block at (k0, k0), in place; *info = k0 + j + 1 at a non-positive pivot
__global__ void __launch_bounds__(kNb * kNb) k_chol_diag(double* __restrict__ L, int N, int k0, int* __restrict__ info) {
  __shared__ double a[kNb][kNb + 1];
  const int nb = min(kNb, N - k0);
  const int r = threadIdx.x / kNb, c = threadIdx.x % kNb;
  a[r][c] = (r < nb && c < nb && c <= r) ? L[(int64_t)(k0 + r) * N + k0 + c] : 0.0;
  __syncthreads();
  for (int j = 0; j < nb; ++j) {
    if (threadIdx.x == 0) {
      const double d = a[j][j];
      if (!(d > 0.0)) { atomicCAS(info, 0, k0 + j + 1); a[j][j] = 1.0; }
      else a[j][j] = sqrt(d);
    }
    __syncthreads();
    if (c == j && r > j && r < nb) a[r][j] /= a[j][j];
    __syncthreads();
    if (c > j && c <= r && r < nb) a[r][c] -= a[r][j] * a[c][j];
    __syncthreads();
  }
  if (r < nb && c < nb) L[(int64_t)(k0 + r) * N + k0 + c] = (c <= r) ? a[r][c] : 0.0;
}

// rows i >= k1:  L[i][k0:k1] <- L[i][k0:k1] L_kk^-T   (one thread per row, L_kk in shared memory)
__global__ void __launch_bounds__(128) k_chol_panel(double* __restrict__ L, int N, int k0) {
  __shared__ double d[kNb][kNb + 1];
  const int k1 = k0 + kNb;
  for (int e = threadIdx.x; e < kNb * kNb; e += 128) d[e / kNb][e % kNb] = L[(int64_t)(k0 + e / kNb) * N + k0 + e % kNb];
  __syncthreads();
  const int i = k1 + blockIdx.x * 128 + threadIdx.x;
  if (i >= N) return;
  double x[kNb];
#pragma unroll
  for (int c = 0; c < kNb; ++c) x[c] = L[(int64_t)i * N + k0 + c];
#pragma unroll
  for (int c = 0; c < kNb; ++c) {           // x L_kk^T = a  ->  x_c = (a_c - sum_{j<c} x_j L_kk[c][j]) / L_kk[c][c]
    double s = x[c];
#pragma unroll
    for (int j = 0; j < c; ++j) s -= x[j] * d[c][j];
    x[c] = s / d[c][c];
  }
#pragma unroll
  for (int c = 0; c < kNb; ++c) L[(int64_t)i * N + k0 + c] = x[c];
}

// trailing update of the lower triangle:  A[i][j] -= sum_{c in [k0, k1)} L[i][c] L[j][c],  i >= j >= k1; 32 x 32 tiles
__global__ void __launch_bounds__(256) k_chol_update(double* __restrict__ L, int N, int k0) {
  __shared__ double pi[kNb][kNb + 1], pj[kNb][kNb + 1];
  const int k1 = k0 + kNb;
  const int bi = blockIdx.y, bj = blockIdx.x;
  if (bj > bi) return;
  const int i0 = k1 + bi * kNb, j0 = k1 + bj * kNb;
  for (int e = threadIdx.x; e < kNb * kNb; e += 256) {
    const int r = e / kNb, c = e % kNb;
    pi[r][c] = (i0 + r < N) ? L[(int64_t)(i0 + r) * N + k0 + c] : 0.0;
    pj[r][c] = (j0 + r < N) ? L[(int64_t)(j0 + r) * N + k0 + c] : 0.0;
  }
  __syncthreads();
  const int c = threadIdx.x % kNb, r4 = threadIdx.x / kNb;      // 8 row groups x 4 rows
#pragma unroll
  for (int rr = 0; rr < 4; ++rr) {
    const int r = r4 * 4 + rr;
    if (i0 + r >= N || j0 + c >= N || j0 + c > i0 + r) continue;
    double s = 0.0;
#pragma unroll
    for (int k = 0; k < kNb; ++k) s = fma(pi[r][k], pj[c][k], s);
    L[(int64_t)(i0 + r) * N + j0 + c] -= s;
  }
}

// block row bi of X = L^-1:  X[bi][bc] = L_bb^-1 ( [bi == bc] I - sum_{bj = bc .. bi-1} L[bi][bj] X[bj][bc] ),  bc <= bi
__global__ void __launch_bounds__(256) k_trinv_row(const double* __restrict__ L, double* __restrict__ X, int N, int bi) {
  __shared__ double la[kNb][kNb + 1], xb[kNb][kNb + 1], acc_s[kNb][kNb + 1];
  const int bc = blockIdx.x;
  const int i0 = bi * kNb, c0 = bc * kNb;
  const int c = threadIdx.x % kNb, r4 = threadIdx.x / kNb;
  double acc[4];
#pragma unroll
  for (int rr = 0; rr < 4; ++rr) acc[rr] = (bi == bc && r4 * 4 + rr == c) ? 1.0 : 0.0;
  for (int bj = bc; bj < bi; ++bj) {
    __syncthreads();
    for (int e = threadIdx.x; e < kNb * kNb; e += 256) {
      const int r = e / kNb, k = e % kNb;
      la[r][k] = (i0 + r < N) ? L[(int64_t)(i0 + r) * N + bj * kNb + k] : 0.0;
      xb[r][k] = X[(int64_t)(bj * kNb + r) * N + c0 + k];
    }
    __syncthreads();
#pragma unroll
    for (int rr = 0; rr < 4; ++rr) {
      const int r = r4 * 4 + rr;
      double s = 0.0;
#pragma unroll
      for (int k = 0; k < kNb; ++k) s = fma(la[r][k], xb[k][c], s);
      acc[rr] -= s;
    }
  }
  __syncthreads();
#pragma unroll
  for (int rr = 0; rr < 4; ++rr) acc_s[r4 * 4 + rr][c] = acc[rr];
  for (int e = threadIdx.x; e < kNb * kNb; e += 256) {
    const int r = e / kNb, k = e % kNb;
    la[r][k] = (i0 + r < N && i0 + k < N) ? L[(int64_t)(i0 + r) * N + i0 + k] : (r == k ? 1.0 : 0.0);
  }
  __syncthreads();
  if (threadIdx.x < kNb) {                  // forward substitution down column c of the right-hand side
    const int cc = threadIdx.x;
    double x[kNb];
#pragma unroll
    for (int r = 0; r < kNb; ++r) {
      double s = acc_s[r][cc];
#pragma unroll
      for (int k = 0; k < r; ++k) s -= la[r][k] * x[k];
      x[r] = s / la[r][r];
    }
#pragma unroll
    for (int r = 0; r < kNb; ++r)
      if (i0 + r < N && c0 + cc < N) X[(int64_t)(i0 + r) * N + c0 + cc] = x[r];
  }
}

__global__ void __launch_bounds__(256) k_zero(double* __restrict__ p, int64_t n) {
  for (int64_t i = (int64_t)blockIdx.x * 256 + threadIdx.x; i < n; i += (int64_t)gridDim.x * 256) p[i] = 0.0;
}

}  // namespace

// S [N][N] (symmetric, only the lower triangle is read) -> L [N][N] (lower, zeros above) and Linv [N][N] = L^-1;
// *info_dev (device int, zeroed here) = 1-based index of the first non-positive pivot, 0 on success.  N % 2 == 0 is
// not required here; N need not be a multiple of the block size.
cudaError_t launch_cholesky_inverse(Op* op, const double* S, int N, double* L, double* Linv, int* info_dev, cudaStream_t st) {
  cudaError_t e;
  if ((e = cudaMemsetAsync(info_dev, 0, sizeof(int), st))) return e;
  const int64_t nn = (int64_t)N * N;
  k_copy_lower<<<(unsigned)((nn + 255) / 256), 256, 0, st>>>(S, L, N);
  op->launches++;
  const int nblk = (N + kNb - 1) / kNb;
  for (int b = 0; b < nblk; ++b) {
    const int k0 = b * kNb, k1 = k0 + kNb;
    k_chol_diag<<<1, kNb * kNb, 0, st>>>(L, N, k0, info_dev);
    op->launches++;
    if (k1 < N) {
      k_chol_panel<<<(unsigned)((N - k1 + 127) / 128), 128, 0, st>>>(L, N, k0);
      const unsigned nt = (unsigned)((N - k1 + kNb - 1) / kNb);
      k_chol_update<<<dim3(nt, nt), 256, 0, st>>>(L, N, k0);
      op->launches += 2;
    }
  }
  k_zero<<<(unsigned)std::min<int64_t>((nn + 255) / 256, 4096), 256, 0, st>>>(Linv, nn);
  op->launches++;
  for (int bi = 0; bi < nblk; ++bi) {
    k_trinv_row<<<(unsigned)(bi + 1), 256, 0, st>>>(L, Linv, N, bi);
    op->launches++;
  }
  return cudaGetLastError();
}

}  // namespace chfsi
