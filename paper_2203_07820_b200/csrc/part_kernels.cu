// Kernels of the cell-partitioned (multi-GPU) form of the filter: the paper's domain decomposition sums the
// rows of the dofs on partition faces over the neighbouring parts once per H~ application, with all vectors of a block in
// one message, optionally in FP32.  A part is an ordinary operator on its own cells
// (chfsi_create_part); what it needs on top are the three memory-bound helpers below.  The exchange itself (NCCL) is the
// caller's: paper_2203_07820_b200/partition.py.
#include "common.h"

namespace chfsi {
namespace {

// buf[s(i)][0..B) = X[rows[i]][0..B), s(i) = slots[i] or i  (U = payload type: the block's own type, or float for the FP32
// boundary traffic)
template <typename T, typename U>
__global__ void __launch_bounds__(256) k_pack_rows(const T* __restrict__ X, int64_t ldx, int B, const int32_t* __restrict__ rows,
                                                   const int32_t* __restrict__ slots, int64_t n_rows, U* __restrict__ buf) {
  const int64_t n = n_rows * B;
  for (int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (int64_t)gridDim.x * blockDim.x) {
    const int64_t r = i / B; const int col = (int)(i - r * B);
    const int64_t sl = slots ? slots[r] : r;
    buf[sl * B + col] = (U)X[(int64_t)rows[r] * ldx + col];
  }
}
// X[rows[i]][0..B) = buf[s(i)][0..B)
template <typename T, typename U>
__global__ void __launch_bounds__(256) k_unpack_rows(const U* __restrict__ buf, const int32_t* __restrict__ rows,
                                                     const int32_t* __restrict__ slots, int64_t n_rows, T* __restrict__ X,
                                                     int64_t ldx, int B) {
  const int64_t n = n_rows * B;
  for (int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (int64_t)gridDim.x * blockDim.x) {
    const int64_t r = i / B; const int col = (int)(i - r * B);
    const int64_t sl = slots ? slots[r] : r;
    X[(int64_t)rows[r] * ldx + col] = (T)buf[sl * B + col];
  }
}
// The accumulate-only form of the exchange (filter in scaled blocks, U14: the cell kernel ADDS this part's
// contribution into the block that holds W_{k-2}): what travels is the part's contribution alone,
//   buf[s(i)] = T[rows[i]] - base[i] + corr X[rows[i]] (1 - owner[i]),
// base = the rows as they were before the kernel ran (nullptr: the kernel stored, base = 0); every part subtracts the
// spectral shift c X once per dof it holds, so the parts that do not own a shared dof put it back: corr = alpha c.
template <typename T, typename U>
__global__ void __launch_bounds__(256) k_pack_rows_delta(const T* __restrict__ Tg, int64_t ldt, const T* __restrict__ base,
                                                         const T* __restrict__ X, int64_t ldx, const uint8_t* __restrict__ owner,
                                                         double corr, int B, const int32_t* __restrict__ rows,
                                                         const int32_t* __restrict__ slots, int64_t n_rows, U* __restrict__ buf) {
  const int64_t n = n_rows * B;
  for (int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (int64_t)gridDim.x * blockDim.x) {
    const int64_t r = i / B; const int col = (int)(i - r * B);
    const int64_t sl = slots ? slots[r] : r;
    double v = (double)Tg[(int64_t)rows[r] * ldt + col];
    if (base) v -= (double)base[i];
    if (!owner[r]) v = fma(corr, (double)X[(int64_t)rows[r] * ldx + col], v);
    buf[sl * B + col] = (U)v;
  }
}
// T[rows[i]] = base[i] + buf[s(i)]   (base = nullptr: 0)
template <typename T, typename U>
__global__ void __launch_bounds__(256) k_unpack_rows_sum(const U* __restrict__ buf, const T* __restrict__ base,
                                                         const int32_t* __restrict__ rows, const int32_t* __restrict__ slots,
                                                         int64_t n_rows, T* __restrict__ Tg, int64_t ldt, int B) {
  const int64_t n = n_rows * B;
  for (int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (int64_t)gridDim.x * blockDim.x) {
    const int64_t r = i / B; const int col = (int)(i - r * B);
    const int64_t sl = slots ? slots[r] : r;
    Tg[(int64_t)rows[r] * ldt + col] = (T)((base ? (double)base[i] : 0.0) + (double)buf[sl * B + col]);
  }
}
// T <- alpha (HX - c X) - beta T: one degree of the scaled three-term recurrence (Eq. 37; U1)
template <typename T>
__global__ void __launch_bounds__(256) k_recurrence(const T* __restrict__ HX, int64_t ldh, const T* __restrict__ X, int64_t ldx,
                                                    T* __restrict__ Tg, int64_t ldt, int64_t n_dofs, int B, double alpha,
                                                    double beta, double c) {
  const int64_t n = n_dofs * B;
  for (int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (int64_t)gridDim.x * blockDim.x) {
    const int64_t g = i / B; const int col = (int)(i - g * B);
    const double h = (double)HX[g * ldh + col], x = (double)X[g * ldx + col];
    const double t = beta != 0.0 ? (double)Tg[g * ldt + col] : 0.0;
    Tg[g * ldt + col] = (T)(alpha * (h - c * x) - beta * t);
  }
}

template <typename T>
cudaError_t pack_t(Op* op, const void* X, int64_t ldx, int64_t B, const int32_t* rows, const int32_t* slots, int64_t n_rows,
                   void* buf, int bp, bool unpack, cudaStream_t st) {
  if (n_rows == 0) return cudaSuccess;
  const unsigned grid = (unsigned)std::min<int64_t>((n_rows * B + 255) / 256, (int64_t)op->n_sm * 16);
  const bool same = bp == (int)(8 * sizeof(T));
  if (!unpack) {
    if (same) k_pack_rows<T, T><<<grid, 256, 0, st>>>((const T*)X, ldx, (int)B, rows, slots, n_rows, (T*)buf);
    else k_pack_rows<T, float><<<grid, 256, 0, st>>>((const T*)X, ldx, (int)B, rows, slots, n_rows, (float*)buf);
  } else {
    if (same) k_unpack_rows<T, T><<<grid, 256, 0, st>>>((const T*)buf, rows, slots, n_rows, (T*)const_cast<void*>(X), ldx, (int)B);
    else k_unpack_rows<T, float><<<grid, 256, 0, st>>>((const float*)buf, rows, slots, n_rows, (T*)const_cast<void*>(X), ldx, (int)B);
  }
  op->launches++;
  return cudaGetLastError();
}

template <typename T>
cudaError_t delta_t(Op* op, void* Tg, int64_t ldt, const void* base, const void* X, int64_t ldx, const uint8_t* owner, double corr,
                    int64_t B, const int32_t* rows, const int32_t* slots, int64_t n_rows, void* buf, int bp, bool unpack,
                    cudaStream_t st) {
  if (n_rows == 0) return cudaSuccess;
  const unsigned grid = (unsigned)std::min<int64_t>((n_rows * B + 255) / 256, (int64_t)op->n_sm * 16);
  const bool same = bp == (int)(8 * sizeof(T));
  if (!unpack) {
    if (same) k_pack_rows_delta<T, T><<<grid, 256, 0, st>>>((const T*)Tg, ldt, (const T*)base, (const T*)X, ldx, owner, corr, (int)B,
                                                           rows, slots, n_rows, (T*)buf);
    else k_pack_rows_delta<T, float><<<grid, 256, 0, st>>>((const T*)Tg, ldt, (const T*)base, (const T*)X, ldx, owner, corr, (int)B,
                                                          rows, slots, n_rows, (float*)buf);
  } else {
    if (same) k_unpack_rows_sum<T, T><<<grid, 256, 0, st>>>((const T*)buf, (const T*)base, rows, slots, n_rows, (T*)Tg, ldt, (int)B);
    else k_unpack_rows_sum<T, float><<<grid, 256, 0, st>>>((const float*)buf, (const T*)base, rows, slots, n_rows, (T*)Tg, ldt, (int)B);
  }
  op->launches++;
  return cudaGetLastError();
}

}  // namespace

cudaError_t launch_rows_delta(Op* op, void* T, int64_t ldt, const void* base, const void* X, int64_t ldx, const uint8_t* owner,
                              double corr, int64_t B, const int32_t* rows, const int32_t* slots, int64_t n_rows, void* buf,
                              int buf_precision, bool unpack, cudaStream_t st) {
  return op->precision == 64
             ? delta_t<double>(op, T, ldt, base, X, ldx, owner, corr, B, rows, slots, n_rows, buf, buf_precision, unpack, st)
             : delta_t<float>(op, T, ldt, base, X, ldx, owner, corr, B, rows, slots, n_rows, buf, buf_precision, unpack, st);
}

cudaError_t launch_pack_rows(Op* op, const void* X, int64_t ldx, int64_t B, const int32_t* rows, const int32_t* slots,
                             int64_t n_rows, void* buf, int buf_precision, bool unpack, cudaStream_t st) {
  return op->precision == 64 ? pack_t<double>(op, X, ldx, B, rows, slots, n_rows, buf, buf_precision, unpack, st)
                             : pack_t<float>(op, X, ldx, B, rows, slots, n_rows, buf, buf_precision, unpack, st);
}

cudaError_t launch_recurrence(Op* op, const void* HX, int64_t ldh, const void* X, int64_t ldx, void* T, int64_t ldt, int64_t B,
                              double alpha, double beta, double c, cudaStream_t st) {
  const unsigned grid = (unsigned)std::min<int64_t>((op->n_dofs * B + 255) / 256, (int64_t)op->n_sm * 16);
  if (op->precision == 64)
    k_recurrence<double><<<grid, 256, 0, st>>>((const double*)HX, ldh, (const double*)X, ldx, (double*)T, ldt, op->n_dofs, (int)B,
                                               alpha, beta, c);
  else
    k_recurrence<float><<<grid, 256, 0, st>>>((const float*)HX, ldh, (const float*)X, ldx, (float*)T, ldt, op->n_dofs, (int)B,
                                              alpha, beta, c);
  op->launches++;
  return cudaGetLastError();
}

}  // namespace chfsi
