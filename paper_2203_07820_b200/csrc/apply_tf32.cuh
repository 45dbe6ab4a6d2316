// FP32 variant of the persistent contraction kernel on the 32-bit tensor pipe (included by apply_kernels.cu).
//
// Same tile protocol as k_apply_dmma_p (tickets in colour order, completion flags, TMA row gather, load-free
// epilogue, -beta Y_{k-2} seeding the accumulators); what differs is the arithmetic of step 2 (Eq. 47,
// PAPER.md:511-513) for FP32-stored matrices and vectors:
//
//   every FP32 operand is split in registers into two TF32 numbers  x = hi + lo,  hi = tf32(x), lo = tf32(x - hi),
//   and  a*b  is accumulated as  a_lo*b_hi + a_hi*b_lo + a_hi*b_hi  with mma.sync.m16n8k8.tf32 (SASS HMMA.1688.F32.TF32)
//   into FP32 accumulators: the dropped a_lo*b_lo term is 2^-22 relative, i.e. FP32-level products at three tensor
//   instructions each.  Single-pass TF32 (10-bit mantissa) cannot hold the 1e-4 tolerance over 30 recurrence steps.
//
// Measured on B200: mma.sync TF32 runs at 277 TFLOP/s (vs 37 TFLOP/s DMMA, 72 TFLOP/s FFMA), so the 3-pass product
// has a ceiling of 92 TFLOP/s of useful FP32 flops; this kernel reaches 39.5 TFLOP/s on config 4 (the operand splits
// and fragment loads share the issue slots) against 30.7 TFLOP/s of the FP64-accumulating default.
//
// OPT-IN ONLY (kernel variant 3): the FP32 accumulator of the tensor pipe truncates instead of rounding to nearest,
// and the partial sums of a stiffness-matrix row are ~|H||x|, so one apply is off by ~2e-6 relative (FP32 FMA:
// 2.5e-7, FP64 accumulation: 4e-8) with a systematic sign.  The filtered block stays inside the 1e-4 tolerance of the
// FP32 variant (1.7e-5 .. 2.9e-5 measured) but the Rayleigh-Ritz values move by up to 4e-5 Ha, outside its 1e-5 Ha
// bound -- so the default FP32 path is k_apply_dmma_p<float>.
//
//   tile   = (cell, 64 columns); 8 warps as 2 (rows) x 4 (columns); warp tile = MT m16-tiles x 2 n8-tiles
//   stream = 16-row K-panels: one bulk copy of the matrix panel + four TMA row gathers of 64 FP32 columns
#pragma once

constexpr int kT3TileN = 64;
constexpr int kT3PanelK = 16;
constexpr int kT3Stages = 4;
constexpr int kT3Ahead = kT3Stages - 2;

__device__ __forceinline__ uint32_t to_tf32(float x) {
  uint32_t r;
  asm("cvt.rna.tf32.f32 %0, %1;" : "=r"(r) : "f"(x));
  return r;
}
__device__ __forceinline__ void split_tf32(float x, uint32_t& hi, uint32_t& lo) {
  hi = to_tf32(x);
  lo = to_tf32(x - __uint_as_float(hi));
}
__device__ __forceinline__ void mma_tf32(float (&c)[4], const uint32_t (&a)[4], uint32_t b0, uint32_t b1) {
  asm("mma.sync.aligned.m16n8k8.row.col.f32.tf32.tf32.f32 {%0,%1,%2,%3}, {%4,%5,%6,%7}, {%8,%9}, {%0,%1,%2,%3};"
      : "+f"(c[0]), "+f"(c[1]), "+f"(c[2]), "+f"(c[3])
      : "r"(a[0]), "r"(a[1]), "r"(a[2]), "r"(a[3]), "r"(b0), "r"(b1));
}
__device__ __forceinline__ float2 ld_cg_f2(const float* p) {
  float2 v;
  asm volatile("ld.global.cg.v2.f32 {%0,%1}, [%2];" : "=f"(v.x), "=f"(v.y) : "l"(p) : "memory");
  return v;
}

inline size_t t3_smem_bytes(const Op* op) {
  return (size_t)kT3Stages * (kT3PanelK * op->lda + kT3PanelK * kT3TileN) * sizeof(float) + 2 * kT3Stages * sizeof(uint64_t) +
         2 * sizeof(long long) + (size_t)op->max_ktot * sizeof(int32_t);
}

template <int MT>
__global__ void __launch_bounds__(kP2Threads, 2) k_apply_tf32_p(ApplyDev<float> a, PersistDev pd,
                                                                const __grid_constant__ CUtensorMap tmX,
                                                                const __grid_constant__ CUtensorMap tmP) {
  extern __shared__ __align__(128) unsigned char smem_raw[];
  const int lda = a.lda;
  const int a_panel_elems = kT3PanelK * lda;
  const int stage_elems = a_panel_elems + kT3PanelK * kT3TileN;
  float* stage0 = reinterpret_cast<float*>(smem_raw);
  uint64_t* full = reinterpret_cast<uint64_t*>(stage0 + kT3Stages * stage_elems);
  uint64_t* empty = full + kT3Stages;
  long long* ticket_s = reinterpret_cast<long long*>(empty + kT3Stages);   // [2]
  int32_t* idx_s = reinterpret_cast<int32_t*>(ticket_s + 2);

  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  const int warp_m = warp >> 2, warp_n = warp & 3;
  const int fg = lane >> 2, ft = lane & 3;   // fragment coordinates: group (row / column n) and thread-in-group (k / column pair)
  const int mc = a.m_cell;
  const int nct = a.n_col_tiles;
  const int n_mtiles = (mc + 15) / 16;
  const int mt0 = warp_m * MT;
  const int nmt = max(0, min(MT, n_mtiles - mt0));
  const float alpha = a.alpha, beta = a.beta;

  if (tid == 0) {
    for (int s = 0; s < kT3Stages; ++s) { mbar_init(&full[s], 1); mbar_init(&empty[s], kP2Threads / 32); }
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    ticket_s[0] = (long long)(atomicAdd(pd.counter, 1ull) - pd.ticket_base);
  }
  __syncthreads();

  uint32_t q0 = 0;   // running panel count: ring slot = q % stages, phase = (q / stages) & 1
  for (int iter = 0;; ++iter) {
    const long long ticket = ticket_s[iter & 1];
    if (ticket >= pd.n_tiles) break;
    const int pos = (int)(ticket / nct), jt = (int)(ticket % nct);
    const int cell = pd.pos_cell[pos];
    const int col0 = jt * kT3TileN;
    const int ncols = min(kT3TileN, a.B - col0);             // multiple of 8
    const int kt = a.ktot[cell];
    const int32_t* gi = a.gidx + a.idx_off[cell];
    const float* M = a.mat + a.mat_off[cell];
    if (tid == 0) ticket_s[(iter + 1) & 1] = (long long)(atomicAdd(pd.counter, 1ull) - pd.ticket_base);
    const bool use_t = (beta != 0.f) && !a.atomic;
    for (int k = tid; k < kt; k += kP2Threads) idx_s[k] = gi[k];
    __syncthreads();

    const int npanel = (kt + kT3PanelK - 1) / kT3PanelK;     // kt is a multiple of 8: the last panel may hold 8 rows
    auto produce = [&](int pj) {
      if (lane != 0) return;
      const uint32_t q = q0 + (uint32_t)pj;
      const int s = (int)(q % kT3Stages);
      mbar_wait(&empty[s], ((q / kT3Stages) & 1u) ^ 1u);
      float* As = stage0 + s * stage_elems;
      float* Xs = As + a_panel_elems;
      const int k0 = pj * kT3PanelK;
      const int rows = min(kT3PanelK, kt - k0);
      const uint32_t a_bytes = (uint32_t)(rows * lda) * 4u;
      mbar_expect_tx(&full[s], a_bytes + (uint32_t)(rows * kT3TileN * 4));
      bulk_g2s(As, M + (int64_t)pj * a_panel_elems, a_bytes, &full[s]);
      for (int r = 0; r < rows; r += 4) {
        const int k = k0 + r;
        tma_gather4(Xs + r * kT3TileN, (k < a.mpad) ? &tmX : &tmP, col0, idx_s[k] & 0x7fffffff, idx_s[k + 1] & 0x7fffffff,
                    idx_s[k + 2] & 0x7fffffff, idx_s[k + 3] & 0x7fffffff, &full[s]);
      }
    };
    if (warp < kT3Ahead && warp < npanel) produce(warp);

    const int nt0 = warp_n * 2;
    const int nnt = max(0, min(2, ncols / 8 - nt0));
    const bool active = (nnt > 0 && nmt > 0);
    // accumulators; those of first-contribution nodes start at (-beta/alpha) Y_{k-2}  (Eq. 37)
    float acc[MT][2][4];
#pragma unroll
    for (int i = 0; i < MT; ++i)
#pragma unroll
      for (int j = 0; j < 2; ++j) acc[i][j][0] = acc[i][j][1] = acc[i][j][2] = acc[i][j][3] = 0.f;
    if (use_t && active) {
      const float nb = -beta / alpha;
#pragma unroll
      for (int i = 0; i < MT; ++i)
#pragma unroll
        for (int h = 0; h < 2; ++h) {
          const int r = (mt0 + i) * 16 + h * 8 + fg;
          const int idx = (i < nmt && r < mc) ? idx_s[r] : 0;
          if (idx < 0) {
            const float* tp = a.Tg + (int64_t)(idx & 0x7fffffff) * a.ldt + col0 + nt0 * 8 + ft * 2;
            const float2 u = ld_cg_f2(tp);
            acc[i][0][2 * h] = u.x; acc[i][0][2 * h + 1] = u.y;
            if (nnt > 1) { const float2 v = ld_cg_f2(tp + 8); acc[i][1][2 * h] = v.x; acc[i][1][2 * h + 1] = v.y; }
          }
        }
#pragma unroll
      for (int i = 0; i < MT; ++i)
#pragma unroll
        for (int j = 0; j < 2; ++j)
#pragma unroll
          for (int e = 0; e < 4; ++e) acc[i][j][e] *= nb;
    }

    for (int pi = 0; pi < npanel; ++pi) {
      const uint32_t q = q0 + (uint32_t)pi;
      const int s = (int)(q % kT3Stages);
      {
        const int pj = pi + kT3Ahead;
        if (pj < npanel && (pj & 7) == warp) produce(pj);
      }
      mbar_wait(&full[s], (q / kT3Stages) & 1u);
      if (active) {
        const float* As = stage0 + s * stage_elems;
        const float* Ap = As + ft * lda + mt0 * 16 + fg;
        const float* Xp = As + a_panel_elems + ft * kT3TileN + nt0 * 8 + fg;
        const int ksteps = min(kT3PanelK, kt - pi * kT3PanelK) / 8;
        for (int ks = 0; ks < ksteps; ++ks) {
          // B fragments (k x n = 8 x 8): b0 = X[k = ft][n = fg], b1 = X[k = ft + 4][n = fg]; columns past ncols are
          // zero-filled by the TMA, so both n-tiles are always computed
          uint32_t bh[2][2], bl[2][2];
#pragma unroll
          for (int j = 0; j < 2; ++j) {
            split_tf32(Xp[j * 8], bh[j][0], bl[j][0]);
            split_tf32(Xp[4 * kT3TileN + j * 8], bh[j][1], bl[j][1]);
          }
#pragma unroll
          for (int i = 0; i < MT; ++i) {
            if (i < nmt) {
              // A fragment (m x k = 16 x 8) of the k-major panel: a0 = A[k = ft][m = fg], a1 = [ft][fg + 8],
              // a2 = [ft + 4][fg], a3 = [ft + 4][fg + 8]
              uint32_t ah[4], al[4];
              split_tf32(Ap[i * 16], ah[0], al[0]);
              split_tf32(Ap[i * 16 + 8], ah[1], al[1]);
              split_tf32(Ap[4 * lda + i * 16], ah[2], al[2]);
              split_tf32(Ap[4 * lda + i * 16 + 8], ah[3], al[3]);
#pragma unroll
              for (int j = 0; j < 2; ++j) {
                mma_tf32(acc[i][j], al, bh[j][0], bh[j][1]);
                mma_tf32(acc[i][j], ah, bl[j][0], bl[j][1]);
                mma_tf32(acc[i][j], ah, bh[j][0], bh[j][1]);
              }
            }
          }
          Ap += 8 * lda;
          Xp += 8 * kT3TileN;
        }
      }
      __syncwarp();
      if (lane == 0) mbar_arrive(&empty[s]);
    }
    q0 += (uint32_t)npanel;

    // ---- epilogue: assembly + recurrence (steps 4-5).  C fragment: rows fg / fg + 8, columns 2 ft + {0, 1}
    if (!a.atomic) {
      const int d1 = pd.dep_ptr[pos + 1];
      for (int d = pd.dep_ptr[pos] + lane; d < d1; d += 32) {
        const uint32_t* f = pd.flags + (int64_t)pd.dep_pos[d] * nct + jt;
        while (ld_acquire_gpu(f) != pd.epoch) __nanosleep(64);
      }
      __syncwarp();
    }
    if (active) {
#pragma unroll
      for (int i = 0; i < MT; ++i)
#pragma unroll
        for (int h = 0; h < 2; ++h) {
          const int r = (mt0 + i) * 16 + h * 8 + fg;
          if (i >= nmt || r >= mc) continue;
          const int idx = idx_s[r];
          float* trow = a.Tg + (int64_t)(idx & 0x7fffffff) * a.ldt + col0 + nt0 * 8 + ft * 2;
          const bool add = a.atomic || idx >= 0;
#pragma unroll
          for (int j = 0; j < 2; ++j) {
            if (j >= nnt) continue;
            const float v0 = alpha * acc[i][j][2 * h], v1 = alpha * acc[i][j][2 * h + 1];
            if (add) {
              atomicAdd(trow + j * 8, v0);
              atomicAdd(trow + j * 8 + 1, v1);
            } else {
              *reinterpret_cast<float2*>(trow + j * 8) = make_float2(v0, v1);
            }
          }
        }
    }
    __threadfence();
    __syncthreads();   // all stores of the tile are done and fenced; idx_s / ticket slot may be reused
    if (tid == 0 && !a.atomic) st_release_gpu(pd.flags + (int64_t)pos * nct + jt, pd.epoch);
  }
}
