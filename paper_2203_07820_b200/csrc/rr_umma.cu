// C = A^T B of two tall FP32 blocks on the 5th-generation tensor cores (tcgen05.mma kind::tf32, accumulators in TMEM):
// the FP32 blocks of the paper's mixed-precision Rayleigh-Ritz products (Sec. 3.2 / 4.4.1: Eq. 38-39, PAPER.md:426-440;
// PAPER.md:564 "FP32 off-diagonal blocks").  Drop-in for k_xty_tf32 (rr_kernels.cu): same split-row partial sums
// Cpart[z][N1][N2] in FP64, same masked reduction; output tiles are 128 x 128 (every MMA reads its operands from shared memory,
// the split warps read and write the same tiles again: at 128 x 64 the kernel was bound by shared-memory bandwidth at 0.27 of
// the TF32 peak, a square tile moves a third less per flop).
//
//   * an FP32 product is a 3xTF32 split, a b ~ a_hi b_lo + a_lo b_hi + a_hi b_hi: hi = x rounded to TF32 (nearest; integer add + mask), lo = x - hi
//     (exact in FP32), both computed by four "split" warps from the tile that the TMA has put into shared memory: hi replaces
//     the tile in place, lo goes to a second tile of the same layout (the swizzle is element-wise transparent);
//   * both operands are MN-major (the stored layout [rows][columns] has the output index fastest and the contraction
//     index = rows).  For MN-major 32-bit operands the tensor core takes ONE shared-memory layout, the 128-byte swizzle with
//     32-byte atoms (SWIZZLE_128B_BASE32B: atoms of 32 columns x 4 rows), which is what a TMA box {32 columns, 32 rows}
//     with CU_TENSOR_MAP_SWIZZLE_128B_ATOM_32B writes; one tcgen05.mma (M = 128, N = 128, K = 8) consumes two such atoms per 32 columns;
//   * the FP32 accumulator of the tensor pipe does not round to nearest, so an accumulation chain is kept to TWO 32-row stages
//     (24 MMAs from zero) in one of two 128-column TMEM buffers; eight epilogue warps drain it (tcgen05.ld) and add the chain
//     sums to FP64 totals in registers (64 per thread: these warps run at 208 registers, setmaxnreg) -- while the next stage's MMAs
//     run into the other buffer;
//   * roles: 8 epilogue warps, 4 split warps, 1 TMA producer warp, 1 MMA warp (one elected lane issues), 2 idle warps that complete
//     the fourth warpgroup for setmaxnreg; 3-stage ring of 64 KB (hi and lo tiles of A and B).
#include <cuda.h>

#include <algorithm>

#include "common.h"

namespace chfsi {
namespace {

constexpr int kUM = 128, kUN = 128, kUK = 32, kUStages = 3;
constexpr int kUEpiWarps = 8, kUSplitWarps = 4;
constexpr int kUThreads = 32 * (kUEpiWarps + kUSplitWarps + 4);                  // + TMA warp, MMA warp, two idle warps (whole warpgroups)
constexpr int kUABytes = kUK * kUM * 4, kUBBytes = kUK * kUN * 4;              // 16 KB, 16 KB
constexpr int kUStageBytes = 2 * (kUABytes + kUBBytes);                          // hi + lo tiles of A and B: 64 KB
constexpr int kUChain = 2;                                                       // stages per accumulation chain in TMEM
constexpr int kURegsEpi = 208, kURegsOther = 48;                                 // setmaxnreg: 8 x 32 x 208 + 8 x 32 x 48 = 64 K registers
constexpr size_t kUSmemBytes = (size_t)kUStages * kUStageBytes + 1024 + 256;

__device__ __forceinline__ uint32_t u_smem(const void* p) { return (uint32_t)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void u_mbar_init(uint64_t* bar, int count) {
  asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(u_smem(bar)), "r"(count));
}
__device__ __forceinline__ void u_mbar_expect_tx(uint64_t* bar, uint32_t bytes) {
  asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(u_smem(bar)), "r"(bytes) : "memory");
}
__device__ __forceinline__ void u_mbar_arrive(uint64_t* bar) {
  asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(u_smem(bar)) : "memory");
}
__device__ __forceinline__ void u_mbar_wait(uint64_t* bar, uint32_t parity) {
  uint32_t done;
  do {
    asm volatile(
        "{\n"
        ".reg .pred p;\n"
        "mbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n"
        "selp.u32 %0, 1, 0, p;\n"
        "}\n"
        : "=r"(done)
        : "r"(u_smem(bar)), "r"(parity)
        : "memory");
  } while (!done);
}
// box {32 columns, 32 rows} of a 2-D FP32 tensor at (column c0, row r0) -> dst (32 rows of 128 bytes, 128B-swizzled)
__device__ __forceinline__ void u_tma_load(void* dst, const CUtensorMap* tm, int c0, int r0, uint64_t* bar) {
  asm volatile("cp.async.bulk.tensor.2d.shared::cluster.global.tile.mbarrier::complete_tx::bytes [%0], [%1, {%3, %4}], [%2];" ::"r"(
                   u_smem(dst)),
               "l"(tm), "r"(u_smem(bar)), "r"(c0), "r"(r0)
               : "memory");
}
// shared-memory matrix descriptor of an MN-major operand in the 128B / 32B-atom swizzle: atoms of 32 columns x 4 rows (512
// bytes); leading byte offset = distance between atoms along MN, stride byte offset = distance between atoms along K
__device__ __forceinline__ uint64_t u_desc(uint32_t smem_addr, uint32_t lbo_bytes, uint32_t sbo_bytes, uint32_t layout_type = 1) {
  uint64_t d = 0;
  d |= (uint64_t)((smem_addr >> 4) & 0x3fff);
  d |= (uint64_t)((lbo_bytes >> 4) & 0x3fff) << 16;
  d |= (uint64_t)((sbo_bytes >> 4) & 0x3fff) << 32;
  d |= (uint64_t)1 << 46;                                  // descriptor version of sm_100
  d |= (uint64_t)layout_type << 61;                        // 1 = SWIZZLE_128B_BASE32B (the one layout of MN-major 32-bit operands), 2 = SWIZZLE_128B
  return d;
}
// instruction descriptor: D = F32, A = B = TF32, both MN-major, N = 64, M = 128, dense, no negation
__host__ __device__ constexpr uint32_t u_idesc(bool a_mn_major) {
  return (1u << 4) | (2u << 7) | (2u << 10) | ((a_mn_major ? 1u : 0u) << 15) | (1u << 16) | ((uint32_t)(kUN >> 3) << 17) |
         ((uint32_t)(kUM >> 4) << 24);
}
__device__ __forceinline__ void u_mma(uint32_t tmem_d, uint64_t adesc, uint64_t bdesc, uint32_t accumulate, uint32_t idesc) {
  asm volatile(
      "{\n"
      ".reg .pred p;\n"
      "setp.ne.b32 p, %4, 0;\n"
      "tcgen05.mma.cta_group::1.kind::tf32 [%0], %1, %2, %3, p;\n"
      "}\n" ::"r"(tmem_d),
      "l"(adesc), "l"(bdesc), "r"(idesc), "r"(accumulate)
      : "memory");
}
__device__ __forceinline__ void u_commit(uint64_t* bar) {
  asm volatile("tcgen05.commit.cta_group::1.mbarrier::arrive::one.shared::cluster.b64 [%0];" ::"r"(u_smem(bar)) : "memory");
}
// 32 consecutive TMEM columns of this thread's lane (32x32b shape: lane = 32 (warp % 4) + lane id)
__device__ __forceinline__ void u_tmem_ld32(uint32_t taddr, float (&v)[32]) {
  uint32_t r[32];
  asm volatile(
      "tcgen05.ld.sync.aligned.32x32b.x32.b32 {%0, %1, %2, %3, %4, %5, %6, %7, %8, %9, %10, %11, %12, %13, %14, %15, %16, %17, "
      "%18, %19, %20, %21, %22, %23, %24, %25, %26, %27, %28, %29, %30, %31}, [%32];"
      : "=r"(r[0]), "=r"(r[1]), "=r"(r[2]), "=r"(r[3]), "=r"(r[4]), "=r"(r[5]), "=r"(r[6]), "=r"(r[7]), "=r"(r[8]), "=r"(r[9]),
        "=r"(r[10]), "=r"(r[11]), "=r"(r[12]), "=r"(r[13]), "=r"(r[14]), "=r"(r[15]), "=r"(r[16]), "=r"(r[17]), "=r"(r[18]),
        "=r"(r[19]), "=r"(r[20]), "=r"(r[21]), "=r"(r[22]), "=r"(r[23]), "=r"(r[24]), "=r"(r[25]), "=r"(r[26]), "=r"(r[27]),
        "=r"(r[28]), "=r"(r[29]), "=r"(r[30]), "=r"(r[31])
      : "r"(taddr)
      : "memory");
  asm volatile("tcgen05.wait::ld.sync.aligned;" ::: "memory");
#pragma unroll
  for (int i = 0; i < 32; ++i) v[i] = __uint_as_float(r[i]);
}

// XZ = false:  Cpart[z] = A^T B over the rows of split z (A, B: [rows][columns], both MN-major; tile = 128 columns of A x 64 of B)
// XZ = true:   Out[g][j] = sum_i Y32[g][i] Z32[i][j] + Y[g][j] zd[j]  (subspace transformation with the FP64 diagonal part,
//              PAPER.md:564): A = Y32 tile of 128 ROWS, K-major (the contraction index i is contiguous: plain 128-byte swizzle),
//              B = Z32 panel, MN-major; blockIdx.x = column tile, blockIdx.y = row block; N1 = number of contraction indices
template <bool XZ>
__global__ void __launch_bounds__(kUThreads, 1) k_umma(const __grid_constant__ CUtensorMap tmA,
                                                       const __grid_constant__ CUtensorMap tmB, int64_t n_rows, int N1, int N2,
                                                       int64_t rows_per_split, int skip_block, int row_block0, int col_block0,
                                                       int lower, double* __restrict__ Cpart, const double* __restrict__ Yd, int64_t ldy,
                                                       const double* __restrict__ zd, int64_t ldo, const int* __restrict__ lower_nonzero) {
  const int i0 = XZ ? 0 : blockIdx.x * kUM, j0 = (XZ ? blockIdx.x : blockIdx.y) * kUN;
  if (!XZ && lower && j0 > i0 + kUM - 1) return;                      // strictly above the diagonal of a Hermitian result
  if (!XZ && skip_block > 0) {                                        // tiles inside an FP64 diagonal block: not ours (k_xty_tf32's rule)
    const int bi0 = (row_block0 + i0) / skip_block, bi1 = (row_block0 + min(i0 + kUM, N1) - 1) / skip_block;
    const int bj0 = (col_block0 + j0) / skip_block, bj1 = (col_block0 + min(j0 + kUN, N2) - 1) / skip_block;
    if (bi0 == bi1 && bj0 == bj1 && bi0 == bj0) return;
  }
  extern __shared__ unsigned char u_raw[];
  unsigned char* sm = reinterpret_cast<unsigned char*>(((uintptr_t)u_raw + 1023) & ~(uintptr_t)1023);   // swizzle atoms: 1024-byte aligned
  uint64_t* bars = reinterpret_cast<uint64_t*>(sm + (size_t)kUStages * kUStageBytes);
  uint64_t* full_raw = bars;                     // [stages] TMA landed
  uint64_t* full_split = bars + kUStages;        // [stages] lo tiles written
  uint64_t* empty = bars + 2 * kUStages;         // [stages] MMAs that read the stage are done
  uint64_t* acc_full = bars + 3 * kUStages;      // [2] accumulator holds a finished stage sum
  uint64_t* acc_empty = acc_full + 2;            // [2] accumulator drained
  uint32_t* tmem_slot = reinterpret_cast<uint32_t*>(acc_empty + 2);
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  const int64_t g0 = XZ ? (int64_t)blockIdx.y * kUM : (int64_t)blockIdx.z * rows_per_split;
  const int64_t g1 = min(n_rows, g0 + (XZ ? (int64_t)kUM : rows_per_split));
  // Y Z with an upper-triangular Z (Z = L^-T): the contraction stops at the last column of the tile (the rest of Z is zero)
  const int nstage = XZ ? (((*lower_nonzero == 0) ? min(N1, j0 + kUN) : N1) + kUK - 1) / kUK : (int)((g1 - g0 + kUK - 1) / kUK);

  if (tid == 0) {
    for (int s = 0; s < kUStages; ++s) { u_mbar_init(full_raw + s, 1); u_mbar_init(full_split + s, kUSplitWarps); u_mbar_init(empty + s, 1); }
    for (int a = 0; a < 2; ++a) { u_mbar_init(acc_full + a, 1); u_mbar_init(acc_empty + a, kUEpiWarps); }
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
  }
  if (warp == kUEpiWarps + kUSplitWarps + 1) {                 // the MMA warp owns the tensor memory: two 128-column accumulators
    asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], %1;" ::"r"(u_smem(tmem_slot)), "n"(2 * kUN) : "memory");
    asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;" ::: "memory");
  }
  asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory");
  __syncthreads();
  asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
  const uint32_t tmem = *reinterpret_cast<volatile uint32_t*>(tmem_slot);

  if (warp < kUEpiWarps) {
    // ---- epilogue warps: lane quarter q = warp % 4 (rows 32 q + lane of the tile), column half h = warp / 4 --------------
    asm volatile("setmaxnreg.inc.sync.aligned.u32 %0;" ::"n"(kURegsEpi));
    const int q = warp & 3, h = warp >> 2;
    constexpr int kHalf = kUN / 2;                                              // 64 columns per thread, FP64 totals in registers
    double tot[kHalf];
#pragma unroll
    for (int j = 0; j < kHalf; ++j) tot[j] = 0.0;
    const int nchain = (nstage + kUChain - 1) / kUChain;
    for (int it = 0; it < nchain; ++it) {
      const int a = it & 1;
      u_mbar_wait(acc_full + a, (uint32_t)(it >> 1) & 1u);
      asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
#pragma unroll
      for (int c = 0; c < kHalf / 32; ++c) {
        float v[32];
        u_tmem_ld32(tmem + ((uint32_t)(32 * q) << 16) + (uint32_t)(a * kUN + kHalf * h + 32 * c), v);
#pragma unroll
        for (int j = 0; j < 32; ++j) tot[32 * c + j] += (double)v[j];           // chain sums (64 rows) are added in FP64
      }
      asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory");
      __syncwarp();
      if (lane == 0) u_mbar_arrive(acc_empty + a);
    }
    if (XZ) {
      const int64_t r = g0 + 32 * q + lane;                                     // Out = FP32 off-diagonal part + FP64 diagonal part
      if (r < n_rows) {
        double* op_ = Cpart + r * ldo + j0 + kHalf * h;
        const double* yp = Yd + r * ldy + j0 + kHalf * h;
#pragma unroll
        for (int j = 0; j < kHalf; ++j)
          if (j0 + kHalf * h + j < N2) op_[j] = fma(yp[j], zd[j0 + kHalf * h + j], tot[j]);
      }
    } else {
      const int r = i0 + 32 * q + lane;
      if (r < N1) {
        double* Cp = Cpart + (int64_t)blockIdx.z * N1 * N2 + (int64_t)r * N2 + j0 + kHalf * h;
#pragma unroll
        for (int j = 0; j < kHalf; ++j)
          if (j0 + kHalf * h + j < N2) Cp[j] = tot[j];
      }
    }
  } else if (warp < kUEpiWarps + kUSplitWarps) {
    asm volatile("setmaxnreg.dec.sync.aligned.u32 %0;" ::"n"(kURegsOther));
    // ---- split warps: lo = x - tf32(x) for the stage's A and B tiles (same offsets: the swizzle is element-wise transparent) ---
    const int st = tid - 32 * kUEpiWarps;
    for (int it = 0; it < nstage; ++it) {
      const int s = it % kUStages;
      unsigned char* base = sm + (size_t)s * kUStageBytes;
      u_mbar_wait(full_raw + s, (uint32_t)(it / kUStages) & 1u);
      // x rounded to TF32 (round to nearest, ties away from zero) as an FP32 value: integer add + mask on the bit pattern
      // (full-rate ALU instructions; cvt.rna.tf32.f32 runs on the slow conversion pipe and made these warps the bottleneck)
      auto rna = [](float x) { return __uint_as_float((__float_as_uint(x) + 0x1000u) & 0xffffe000u); };
      auto split = [&](float4* src, float4* dst, int n4, int t0) {     // src <- hi = tf32(x), dst <- lo = x - hi (exact)
        for (int e = t0; e < n4; e += 32 * kUSplitWarps) {
          const float4 x = src[e];
          float4 hv, l;
          hv.x = rna(x.x); hv.y = rna(x.y); hv.z = rna(x.z); hv.w = rna(x.w);
          l.x = x.x - hv.x; l.y = x.y - hv.y; l.z = x.z - hv.z; l.w = x.w - hv.w;
          src[e] = hv;
          dst[e] = l;
        }
      };
      split(reinterpret_cast<float4*>(base), reinterpret_cast<float4*>(base + kUABytes), kUABytes / 16, st);
      split(reinterpret_cast<float4*>(base + 2 * kUABytes), reinterpret_cast<float4*>(base + 2 * kUABytes + kUBBytes),
            kUBBytes / 16, st);
      asm volatile("fence.proxy.async.shared::cta;" ::: "memory");   // generic writes of the lo tiles before the tensor core reads them
      __syncwarp();
      if (lane == 0) u_mbar_arrive(full_split + s);
    }
  } else {
    asm volatile("setmaxnreg.dec.sync.aligned.u32 %0;" ::"n"(kURegsOther));   // warps 12 .. 15: one warpgroup (TMA, MMA, two idle)
    if (warp == kUEpiWarps + kUSplitWarps) {
    // ---- TMA producer ---------------------------------------------------------------------------------------------------
    if (lane == 0) {
      for (int it = 0; it < nstage; ++it) {
        const int s = it % kUStages;
        unsigned char* base = sm + (size_t)s * kUStageBytes;
        u_mbar_wait(empty + s, ((uint32_t)(it / kUStages) & 1u) ^ 1u);
        u_mbar_expect_tx(full_raw + s, (uint32_t)(kUABytes + kUBBytes));
        const int r0 = XZ ? it * kUK : (int)(g0 + (int64_t)it * kUK);             // first contraction index of the stage
        if (XZ) {
          u_tma_load(base, &tmA, r0, (int)g0, full_raw + s);                     // 128 rows x 32 contraction indices (K-major)
        } else {
#pragma unroll
          for (int m = 0; m < kUM / 32; ++m) u_tma_load(base + m * 4096, &tmA, i0 + 32 * m, r0, full_raw + s);
        }
#pragma unroll
        for (int m = 0; m < kUN / 32; ++m) u_tma_load(base + 2 * kUABytes + m * 4096, &tmB, j0 + 32 * m, r0, full_raw + s);
      }
    }
    } else if (warp == kUEpiWarps + kUSplitWarps + 1) {
    // ---- MMA warp: one lane issues; per stage 4 k-atoms x (hi lo + lo hi + hi hi) from zero into accumulator it & 1 --------
    if (lane == 0) {
      for (int it = 0; it < nstage; ++it) {
        const int s = it % kUStages, ch = it / kUChain, a = ch & 1;
        const bool first = it % kUChain == 0, last = it % kUChain == kUChain - 1 || it == nstage - 1;
        const uint32_t sbase = u_smem(sm + (size_t)s * kUStageBytes);
        if (first) u_mbar_wait(acc_empty + a, ((uint32_t)(ch >> 1) & 1u) ^ 1u);
        u_mbar_wait(full_split + s, (uint32_t)(it / kUStages) & 1u);
        asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
        const uint32_t d = tmem + (uint32_t)(a * kUN);
#pragma unroll
        for (int ka = 0; ka < kUK / 8; ++ka) {
          // A: MN-major atoms (X^T Y), or K-major rows of 128 bytes in 8-row groups of 1024 bytes, 32 bytes per k-step (Y Z)
          const uint64_t ahi = XZ ? u_desc(sbase + ka * 32, 16, 1024, 2) : u_desc(sbase + ka * 1024, 4096, 512);
          const uint64_t alo = XZ ? u_desc(sbase + kUABytes + ka * 32, 16, 1024, 2) : u_desc(sbase + kUABytes + ka * 1024, 4096, 512);
          const uint64_t bhi = u_desc(sbase + 2 * kUABytes + ka * 1024, 4096, 512);
          const uint64_t blo = u_desc(sbase + 2 * kUABytes + kUBBytes + ka * 1024, 4096, 512);
          u_mma(d, ahi, blo, (ka > 0 || !first) ? 1u : 0u, u_idesc(!XZ));
          u_mma(d, alo, bhi, 1u, u_idesc(!XZ));
          u_mma(d, ahi, bhi, 1u, u_idesc(!XZ));
        }
        u_commit(empty + s);          // the stage may be refilled once these MMAs have read it
        if (last) u_commit(acc_full + a);   // ... and the accumulator holds the sum of the chain
      }
    }
    }
  }
  asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory");
  __syncthreads();
  if (warp == kUEpiWarps + kUSplitWarps + 1)
    asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, %1;" ::"r"(tmem), "n"(2 * kUN) : "memory");
}

using UEncodeFn = CUresult (*)(CUtensorMap*, CUtensorMapDataType, cuuint32_t, void*, const cuuint64_t*, const cuuint64_t*,
                               const cuuint32_t*, const cuuint32_t*, CUtensorMapInterleave, CUtensorMapSwizzle,
                               CUtensorMapL2promotion, CUtensorMapFloatOOBfill);
UEncodeFn u_encode_fn() {
  static UEncodeFn fn = [] {
    void* p = nullptr;
    cudaDriverEntryPointQueryResult q;
    if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &p, cudaEnableDefault, &q) != cudaSuccess || q != cudaDriverEntryPointSuccess)
      p = nullptr;
    return reinterpret_cast<UEncodeFn>(p);
  }();
  return fn;
}
// FP32 block [rows][ld] restricted to `cols` columns; box = 32 columns x 32 rows, 128-byte swizzle, zero fill outside
// (k_major: box = 32 columns x 128 rows in the plain 128-byte swizzle: the K-major A operand of the Y Z product)
bool u_make_map(CUtensorMap* tm, const float* base, int64_t rows, int64_t cols, int64_t ld, bool k_major = false) {
  UEncodeFn enc = u_encode_fn();
  if (!enc || rows < 1 || cols < 1 || (ld * 4) % 16 != 0 || (uintptr_t)base % 16 != 0) return false;
  const cuuint64_t dims[2] = {(cuuint64_t)cols, (cuuint64_t)rows};
  const cuuint64_t strides[1] = {(cuuint64_t)ld * 4};
  const cuuint32_t box[2] = {32, (cuuint32_t)(k_major ? kUM : kUK)};
  const cuuint32_t estr[2] = {1, 1};
  return enc(tm, CU_TENSOR_MAP_DATA_TYPE_FLOAT32, 2, const_cast<float*>(base), dims, strides, box, estr, CU_TENSOR_MAP_INTERLEAVE_NONE,
             k_major ? CU_TENSOR_MAP_SWIZZLE_128B : CU_TENSOR_MAP_SWIZZLE_128B_ATOM_32B, CU_TENSOR_MAP_L2_PROMOTION_L2_256B,
             CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE) == CUDA_SUCCESS;
}

}  // namespace

cudaError_t init_umma_kernels() {
  cudaError_t e = cudaFuncSetAttribute(k_umma<false>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)kUSmemBytes);
  if (e != cudaSuccess) return e;
  return cudaFuncSetAttribute(k_umma<true>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)kUSmemBytes);
}

// Row splits of the X^T Y product for this kernel: one CTA per SM, equal work per CTA, so the split count is the one whose CTA
// count (tiles that are not skipped x splits) fills its last wave best, among 2 .. 8 waves and >= 2,048 rows per split.
void umma_xty_plan(int n_sm, int64_t n_rows, int N1, int N2, int skip_block, int row_block0, int col_block0, int lower,
                   int* n_split, int64_t* rows_per_split) {
  int tiles = 0;
  for (int i0 = 0; i0 < N1; i0 += kUM)
    for (int j0 = 0; j0 < N2; j0 += kUN) {
      bool skip = lower && j0 > i0 + kUM - 1;
      if (!skip && skip_block > 0) {
        const int bi0 = (row_block0 + i0) / skip_block, bi1 = (row_block0 + std::min(i0 + kUM, N1) - 1) / skip_block;
        const int bj0 = (col_block0 + j0) / skip_block, bj1 = (col_block0 + std::min(j0 + kUN, N2) - 1) / skip_block;
        skip = bi0 == bi1 && bj0 == bj1 && bi0 == bj0;
      }
      tiles += skip ? 0 : 1;
    }
  tiles = std::max(tiles, 1);
  const int ns_max = (int)std::max<int64_t>(1, n_rows / 2048);
  const int ns_lo = std::min(ns_max, std::max(1, (2 * n_sm + tiles - 1) / tiles));
  const int ns_hi = std::min(ns_max, std::max(ns_lo, 8 * n_sm / tiles));
  int best_ns = ns_lo;
  double best = 0.0;
  for (int ns = ns_lo; ns <= ns_hi; ++ns) {
    const int64_t ctas = (int64_t)tiles * ns;
    const double eff = (double)ctas / (double)(((ctas + n_sm - 1) / n_sm) * n_sm);
    if (eff > best + 1e-9) { best = eff; best_ns = ns; }
  }
  *rows_per_split = ((n_rows + best_ns - 1) / best_ns + kUK - 1) / kUK * kUK;
  *n_split = (int)((n_rows + *rows_per_split - 1) / *rows_per_split);
}

// Cpart[z][N1][N2] (FP64) = per-split sums of A^T B; returns false when the tensor maps cannot be built (caller falls back)
bool launch_xty_umma(const float* A, int64_t lda, const float* B, int64_t ldb, int64_t n_rows, int N1, int N2, int n_split,
                     int64_t rows_per_split, int skip_block, int row_block0, int col_block0, int lower, double* Cpart,
                     cudaStream_t st) {
  CUtensorMap tmA, tmB;
  if (!u_make_map(&tmA, A, n_rows, N1, lda) || !u_make_map(&tmB, B, n_rows, N2, ldb)) return false;
  dim3 grid((unsigned)((N1 + kUM - 1) / kUM), (unsigned)((N2 + kUN - 1) / kUN), (unsigned)n_split);
  k_umma<false><<<grid, kUThreads, kUSmemBytes, st>>>(tmA, tmB, n_rows, N1, N2, rows_per_split, skip_block, row_block0, col_block0, lower,
                                                      Cpart, nullptr, 0, nullptr, 0, nullptr);
  return true;
}

// Out[g][j] = sum_i Y32[g][i] Z32[i][j] (3xTF32) + Y[g][j] zd[j] (FP64), g < n_rows, i < N, j < N2; false: no tensor maps
bool launch_xz_umma(const float* Y32, int64_t ldy32, const float* Z32, int64_t ldz32, const double* Y, int64_t ldy, const double* zd,
                    int64_t n_rows, int N, int N2, double* Out, int64_t ldo, const int* lower_nonzero, cudaStream_t st) {
  CUtensorMap tmA, tmB;
  if (!u_make_map(&tmA, Y32, n_rows, N, ldy32, true) || !u_make_map(&tmB, Z32, N, N2, ldz32)) return false;
  dim3 grid((unsigned)((N2 + kUN - 1) / kUN), (unsigned)((n_rows + kUM - 1) / kUM));
  k_umma<true><<<grid, kUThreads, kUSmemBytes, st>>>(tmA, tmB, n_rows, N, N2, 0, 0, 0, 0, 0, Out, Y, ldy, zd, ldo, lower_nonzero);
  return true;
}

}  // namespace chfsi
