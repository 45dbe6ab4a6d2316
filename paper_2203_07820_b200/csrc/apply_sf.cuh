// Sum-factorised (matrix-free) variant of the fused H~ application + recurrence update, FE degree p <= 6.
// Included by apply_kernels.cu (uses its mbarrier / TMA / flag helpers and the ticket protocol of k_apply_dmma_p).
//
// north_star: the per-cell contraction H^e X^e runs "as FP64 tensor-core batched GEMM ... or sum-factorised where
// measurement says so".  On B200 the FP64 tensor pipe (DMMA) is no faster than the FP64 ALUs (both 37 TFLOP/s, and
// they are ONE pipe: mixed DMMA + DFMA streams never exceed that sum), so the operation count decides.  The dense
// product costs 2 M_cell^2 = 235 kflop per cell and vector at p = 6; the tensor-product structure of the basis,
// N_l(q) = phi_a(qa) phi_b(qb) phi_c(qc) (spectral FE on GLL nodes), gives the same result with 102 kflop:
//
//   u_l = s_l x_g(l)                                              extraction + M^-1/2 (Eq. 47 step i; Eq. 34)
//   u^(q) = sum_l N_l(q) u_l                                      three 1-D contractions with Phi [nq1 x n1]
//   d_e u^(q), e = x,y,z                                          1-D collocation derivative Dh [nq1 x nq1] on the Gauss grid
//                                                                  (exact: u^ has degree p < nq1 per direction)
//   v(q) = W0(q) u^(q),  g_d(q) = sum_e G_de(q) d_e u^(q)          W0 = w detJ V_eff, G = 1/2 w detJ J^-1 J^-T: exactly the
//                                                                  quadrature of Eq. 30 terms 1-2 / Eq. 40
//   w(q) = v(q) + sum_d (Dh_d^T g_d)(q);   y_l = sum_q N_l(q) w(q)  the transposes of the above
//   T[g(l)] (+)= alpha (s_l y_l + (C~^c P)_l - c x_g [first]) - beta T[g]   assembly, Alg. 4 step 5, recurrence (as k_apply_dmma_p)
//
// Mapping (one warp = two adjacent columns at a time, so that every 1-D matrix entry and every field value that is
// loaded serves two columns and two independent dependency chains are in flight; lane = 4 g + t):
//   * a 1-D contraction over the index that is spread over t runs as two m8n8k4 DMMAs per 8 x 8 slab; chaining
//     "matrix x data" (data = B operand, read from shared memory) with "data x matrix" (data = A operand = the C
//     fragment of the previous product: with the contraction index ordered (2t, 2t+1) the C fragment IS the A fragment
//     pair) applies two directions without moving data; the third direction lives in the lane's registers and is plain
//     DFMA with the 1-D matrices as constant-bank operands; the x-direction of the gradient and of the final
//     interpolation needs the slab transposed, which is one trip through a per-warp scratch slab in shared memory.
//   * canonical register layout of a field on the Gauss grid: lane (g, t) holds (qa = g, qb = 2t + {0, 1}) for all qc.
//   * tile = (cell, 16 FP64 | 32 FP32 columns); its rows are gathered by TMA tile::gather4 with SWIZZLE_128B (row =
//     128 bytes), so that the B-fragment loads (32 lanes = 32 different rows, one column) spread over the banks; the
//     result of a column overwrites the column in place.  The CTA then assembles the tile with the thread mapping of an
//     m8n8 C fragment (8 rows x 64 bytes per store instruction); the projector term C~^c P (Alg. 4 step 5)
//     is one more k = 8 DMMA per 8 x 8 block of the tile, accumulated onto it before the scatter.
#pragma once

constexpr int kSfThreads = 128;
constexpr int kSfWarps = kSfThreads / 32;
constexpr int kSfScrPitch = 10;                  // doubles per row of a scratch slab (bank-conflict-free, 16-byte rows)
constexpr int kSfScrSlab = 8 * kSfScrPitch;
constexpr int kSfCrowChunk = 8;                  // projector columns of a cell staged in shared memory for the assembly
constexpr int kSfMaxProj = 16;                   // projectors touching one cell (more: the dense kernel takes the operator)
template <typename S> __host__ __device__ constexpr int sf_cpc() { return 16 / (int)sizeof(S); }        // columns per 16-byte chunk
template <typename S> __host__ __device__ constexpr int sf_tile_cols() { return 8 * sf_cpc<S>(); }      // 16 | 32

// 1-D tables of the degrees in use, zero-padded to 8 x 8: Phi[q][i] = l_i(x_q), Dh[q'][q] = (d/dx) lhat_q (x_q')
__constant__ double c_sf_phi[7][64];
__constant__ double c_sf_dhat[7][64];

struct SfDev {
  const double* __restrict__ coef;           // [n_cells][nq1][7][32 lanes][2]: W0, Gxx, Gxy, Gxz, Gyy, Gyz, Gzz at the lane's points
  const double* __restrict__ sloc;           // [n_cells][mpad]  M^-1/2 at the nodes of the cell
  const double* __restrict__ crows;          // [nnz_cell_proj][mpad]  s_l C^c_{l,j} (rows padded with zeros)
  const int64_t* __restrict__ cell_proj_ptr; // [n_cells + 1]
  double cshift;                             // spectral shift c of the running filter (0 for apply_H)
  int zero;                                  // 0 (k_apply_sf_ws: keeps the 1-D table addresses out of ptxas's hoisting)
};

template <int P, typename S>
size_t sf_smem_bytes(const Op* op) {
  constexpr int nq1 = P + 2;
  size_t b = (size_t)op->mpad * 128;                                   // tile rows
  b += (size_t)nq1 * 7 * 64 * sizeof(double);                          // coefficient fields of the cell
  b += (size_t)kSfWarps * 4 * kSfScrSlab * sizeof(double);             // per-warp transposition scratch: 2 slabs x 2 columns
  b += (size_t)op->mpad * 16;                                          // {s_l, c or 0} per node
  b += (size_t)2 * kSfMaxProj * sf_tile_cols<S>() * sizeof(double);    // rows of P for the cell (this tile, next tile)
  b += (size_t)2 * (op->mpad + kSfMaxProj) * sizeof(int32_t) + 64;     // index lists (this tile, next tile), barriers, tickets
  return b;
}

// the two adjacent columns (2 pp, 2 pp + 1) of tile row l: one 16-byte (FP64) / 8-byte (FP32) shared-memory access
template <typename S> __device__ __forceinline__ uint32_t sf_pair_off(int l, int pp);
template <> __device__ __forceinline__ uint32_t sf_pair_off<double>(int l, int pp) {
  return (uint32_t)l * 128u + ((uint32_t)(pp ^ (l & 7)) << 4);
}
template <> __device__ __forceinline__ uint32_t sf_pair_off<float>(int l, int pp) {
  return (uint32_t)l * 128u + ((uint32_t)((pp >> 1) ^ (l & 7)) << 4) + (uint32_t)(pp & 1) * 8u;
}
__device__ __forceinline__ double2 sf_ld_pair(const double* p) { return *reinterpret_cast<const double2*>(p); }
__device__ __forceinline__ double2 sf_ld_pair(const float* p) {
  const float2 v = *reinterpret_cast<const float2*>(p);
  return make_double2((double)v.x, (double)v.y);
}
__device__ __forceinline__ void sf_st_pair(double* p, double a, double b) { *reinterpret_cast<double2*>(p) = make_double2(a, b); }
__device__ __forceinline__ void sf_st_pair(float* p, double a, double b) { *reinterpret_cast<float2*>(p) = make_float2((float)a, (float)b); }
__device__ __forceinline__ double2 sf_ldg_pair(const double* p) { return ld_cg_d2(p); }
__device__ __forceinline__ double2 sf_ldg_pair(const float* p) { return ld_cg_pair(p); }

template <int P, typename S>
__global__ void __launch_bounds__(kSfThreads, 2) k_apply_sf(ApplyDev<S> a, SfDev sf, PersistDev pd,
                                                            const __grid_constant__ CUtensorMap tmX) {
  constexpr int n1 = P + 1, nq1 = P + 2, nn = n1 * n1, mc = n1 * nn;
  constexpr int TN = sf_tile_cols<S>();
  constexpr int NT = TN / 8;                               // 8-column blocks of the tile
  constexpr int coef_elems = nq1 * 7 * 64;
  extern __shared__ __align__(1024) unsigned char smem_dyn[];
  const int mpad = a.mpad;
  unsigned char* xt = smem_dyn;                                                     // [mpad][128 B], swizzled (1024-byte aligned)
  double* coef_s = reinterpret_cast<double*>(xt + (size_t)mpad * 128);              // [nq1][7][32][2]
  double* scr_all = coef_s + coef_elems;                                            // [warps][4][kSfScrSlab]
  double2* tab_s = reinterpret_cast<double2*>(scr_all + kSfWarps * 4 * kSfScrSlab); // [mpad]
  double* Ps_all = reinterpret_cast<double*>(tab_s + mpad);                         // [2][kSfMaxProj][TN]
  uint64_t* bar = reinterpret_cast<uint64_t*>(Ps_all + 2 * kSfMaxProj * TN);       // [2]: tile data, projector columns
  long long* ticket_s = reinterpret_cast<long long*>(bar + 2);                      // [2]
  int32_t* idx_all = reinterpret_cast<int32_t*>(ticket_s + 2);                      // [2][mpad + kSfMaxProj]

  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  const int g = lane >> 2, t = lane & 3;
  const int nct = a.n_col_tiles;
  // scratch slabs of this warp: [buffer A | B][column u]; element (row, col) of a slab at row * pitch + col
  double* scrA = scr_all + warp * 4 * kSfScrSlab;
  double* scrB = scrA + 2 * kSfScrSlab;
  const int so_w = g * kSfScrPitch + 2 * t;                   // where this lane writes its C-fragment pair (row g, cols 2t, 2t+1)
  const int so_r0 = t * kSfScrPitch + g, so_r1 = (4 + t) * kSfScrPitch + g;   // B fragments: (k = 4s + t, n = g)

  // constant fragments of the 1-D matrices (k-step s: contraction index 4s + t for "matrix x data", 2t + s for
  // "data x matrix")
  double fPhiA[2], fPhiB[2], fDA[2], fDB[2], fDtA[2], fDtB[2], fPhiTA[2], fPhiTB[2];
#pragma unroll
  for (int s = 0; s < 2; ++s) {
    fPhiA[s] = c_sf_phi[P][g * 8 + 4 * s + t];           // Phi[qa = g][a = 4s + t]
    fPhiB[s] = c_sf_phi[P][g * 8 + 2 * t + s];           // Phi[qb = g][b = 2t + s]
    fDA[s] = c_sf_dhat[P][g * 8 + 4 * s + t];            // Dh[qa' = g][qa = 4s + t]
    fDB[s] = c_sf_dhat[P][g * 8 + 2 * t + s];            // Dh[qb' = g][qb = 2t + s]
    fDtA[s] = c_sf_dhat[P][(4 * s + t) * 8 + g];         // Dh[qa = 4s + t][qa'' = g]
    fDtB[s] = c_sf_dhat[P][(2 * t + s) * 8 + g];         // Dh[qb = 2t + s][qb'' = g]
    fPhiTA[s] = c_sf_phi[P][(4 * s + t) * 8 + g];        // Phi[qa = 4s + t][a = g]
    fPhiTB[s] = c_sf_phi[P][(2 * t + s) * 8 + g];        // Phi[qb = 2t + s][b = g]
  }

  if (tid == 0) {
    mbar_init(bar, 1);
    mbar_init(bar + 1, 1);
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    ticket_s[0] = (long long)(atomicAdd(pd.counter, 1ull) - pd.ticket_base);
  }
  __syncthreads();

  // Small per-tile data: index list (dofs of the cell's nodes, then its projector ids), {M^-1/2, shift} per node, the
  // rows of P of the cell's projectors.  Those of the NEXT tile are fetched into registers at the start of the assembly
  // of the current tile and stored at its end, and the next tile's rows and fields are requested right after the
  // completion flag is released: the next tile starts with a wait on the copies only.
  constexpr int kIdxStride = (mc + 7) / 8 * 8 + kSfMaxProj;
  constexpr int kIdxPer = (kIdxStride + kSfThreads - 1) / kSfThreads;
  constexpr int kPsPer = kSfMaxProj * TN / kSfThreads;
  int idx_pre[kIdxPer];
  double sl_pre[kIdxPer], p_pre[kPsPer];
  auto load_small = [&](long long ticket_l, int& cell_l, int& col0_l) {
    cell_l = pd.pos_cell[(int)(ticket_l / nct)];
    col0_l = (int)(ticket_l % nct) * TN;
    const int32_t* gi_l = a.gidx + a.idx_off[cell_l];
    const int np_l = (int)(sf.cell_proj_ptr[cell_l + 1] - sf.cell_proj_ptr[cell_l]);
    const int ncols_l = min(TN, a.B - col0_l);
#pragma unroll
    for (int i = 0; i < kIdxPer; ++i) {
      const int k = tid + i * kSfThreads;
      idx_pre[i] = (k < mpad + np_l) ? gi_l[k] : 0;
      sl_pre[i] = (k < mc) ? sf.sloc[(int64_t)cell_l * mpad + k] : 0.0;
    }
#pragma unroll
    for (int i = 0; i < kPsPer; ++i) {
      const int e = tid + i * kSfThreads, jj = e / TN, cc = e % TN;
      p_pre[i] = (jj < np_l && cc < ncols_l) ? (double)a.P[(int64_t)gi_l[mpad + jj] * a.ldp + col0_l + cc] : 0.0;
    }
  };
  auto store_small = [&](int32_t* idx_l, double* Ps_l) {
#pragma unroll
    for (int i = 0; i < kIdxPer; ++i) {
      const int k = tid + i * kSfThreads;
      if (k < kIdxStride) idx_l[k] = idx_pre[i];
      if (k < mpad) tab_s[k] = make_double2(sl_pre[i], (idx_pre[i] < 0) ? sf.cshift : 0.0);
    }
#pragma unroll
    for (int i = 0; i < kPsPer; ++i) Ps_l[tid + i * kSfThreads] = p_pre[i];
  };
  auto issue_tile = [&](const int32_t* idx_l, int cell_l, int col0_l) {      // warp 0, all lanes
    if (lane == 0) {
      mbar_expect_tx(bar, (uint32_t)mpad * 128u + (uint32_t)(coef_elems * sizeof(double)));
      bulk_g2s(coef_s, sf.coef + (int64_t)cell_l * coef_elems, (uint32_t)(coef_elems * sizeof(double)), bar);
    }
    __syncwarp();
    for (int r4 = lane; r4 < mpad / 4; r4 += 32)
      tma_gather4(xt + (size_t)r4 * 512, &tmX, col0_l, idx_l[4 * r4] & 0x7fffffff, idx_l[4 * r4 + 1] & 0x7fffffff,
                  idx_l[4 * r4 + 2] & 0x7fffffff, idx_l[4 * r4 + 3] & 0x7fffffff, bar);
  };
  if (ticket_s[0] < pd.n_tiles) {
    int cell_f, col0_f;
    load_small(ticket_s[0], cell_f, col0_f);
    store_small(idx_all, Ps_all);
    __syncthreads();
    if (warp == 0) issue_tile(idx_all, cell_f, col0_f);
  }

  uint32_t phase = 0, phase_c = 0;   // parities of the two barriers (tile data / projector columns)
  for (int iter = 0;; ++iter) {
    if (ticket_s[iter & 1] >= pd.n_tiles) break;
    {
    const int ncols = min(TN, a.B - (int)(ticket_s[iter & 1] % nct) * TN);   // even: B is a multiple of the 16-byte chunk
    if (tid == 0) ticket_s[(iter + 1) & 1] = (long long)(atomicAdd(pd.counter, 1ull) - pd.ticket_base);
    mbar_wait(bar, phase);

    // ------------------------------------------------------------------------------------------------------------
    // two adjacent columns (2 pp, 2 pp + 1) at a time per warp; arrays are [..][u = column][e = second point / node]
    // ------------------------------------------------------------------------------------------------------------
    for (int pp = warp; 2 * pp < ncols; pp += kSfWarps) {
      double uh[nq1][2][2], w[nq1][2][2];
      {
        // ---- forward interpolation: u^ = (Phi x Phi x Phi) u ----------------------------------------------------
        double T2[n1][2][2];
        {
          double d[n1][2][2];
#pragma unroll
          for (int s = 0; s < 2; ++s) {
            double bv[n1][2];
            const int ai = 4 * s + t;
            const bool ok = (ai < n1) && (g < n1);
#pragma unroll
            for (int c = 0; c < n1; ++c) {
              const int l = ai + n1 * g + nn * c;
              bv[c][0] = bv[c][1] = 0.0;
              if (ok) {
                const double2 x2 = sf_ld_pair(reinterpret_cast<const S*>(xt + sf_pair_off<S>(l, pp)));
                const double sl = tab_s[l].x;
                bv[c][0] = x2.x * sl; bv[c][1] = x2.y * sl;
              }
            }
#pragma unroll
            for (int c = 0; c < n1; ++c)
#pragma unroll
              for (int u = 0; u < 2; ++u) {
                if (s == 0) d[c][u][0] = d[c][u][1] = 0.0;
                dmma884(d[c][u][0], d[c][u][1], fPhiA[s], bv[c][u]);       // T1[c][b][qa] = sum_a Phi[qa][a] u[c][b][a]
              }
          }
#pragma unroll
          for (int c = 0; c < n1; ++c)
#pragma unroll
            for (int u = 0; u < 2; ++u) T2[c][u][0] = T2[c][u][1] = 0.0;
#pragma unroll
          for (int s = 0; s < 2; ++s)
#pragma unroll
            for (int c = 0; c < n1; ++c)
#pragma unroll
              for (int u = 0; u < 2; ++u)
                dmma884(T2[c][u][0], T2[c][u][1], d[c][u][s], fPhiB[s]);    // T2[c][qb][qa] = sum_b T1 Phi[qb][b]
        }
#pragma unroll
        for (int q = 0; q < nq1; ++q)
#pragma unroll
          for (int u = 0; u < 2; ++u) uh[q][u][0] = uh[q][u][1] = w[q][u][0] = w[q][u][1] = 0.0;
        // third direction in the lane's registers, outer-product order: 4 nq1 independent accumulators
#pragma unroll
        for (int c = 0; c < n1; ++c)
#pragma unroll
          for (int q = 0; q < nq1; ++q) {
            const double ph = c_sf_phi[P][q * 8 + c];
#pragma unroll
            for (int u = 0; u < 2; ++u) {
              uh[q][u][0] = fma(ph, T2[c][u][0], uh[q][u][0]);
              uh[q][u][1] = fma(ph, T2[c][u][1], uh[q][u][1]);
            }
          }
      }

      // ---- Gauss grid, slab by slab: gradient, metric / potential, transposed gradient -----------------------------
      // buffer A carries the slab of u^ (read back with qa as the contraction index for d_x), buffer B the slab of g_x,
      // whose transposed derivative is applied one iteration later.
#pragma unroll
      for (int q = 0; q <= nq1; ++q) {
        double b0[2], b1[2], c0[2], c1[2];
        if (q < nq1) {
#pragma unroll
          for (int u = 0; u < 2; ++u)
            *reinterpret_cast<double2*>(scrA + u * kSfScrSlab + so_w) = make_double2(uh[q][u][0], uh[q][u][1]);
        }
        __syncwarp();
        if (q < nq1) {
#pragma unroll
          for (int u = 0; u < 2; ++u) { b0[u] = scrA[u * kSfScrSlab + so_r0]; b1[u] = scrA[u * kSfScrSlab + so_r1]; }
        }
        if (q > 0) {
#pragma unroll
          for (int u = 0; u < 2; ++u) { c0[u] = scrB[u * kSfScrSlab + so_r0]; c1[u] = scrB[u * kSfScrSlab + so_r1]; }
        }
        __syncwarp();                                                  // both buffers may be rewritten
        if (q > 0) {
#pragma unroll
          for (int u = 0; u < 2; ++u) {
            dmma884(w[q - 1][u][0], w[q - 1][u][1], fDtA[0], c0[u]);   // += sum_qa Dh[qa][qa''] g_x[qa][qb]   (slab q - 1)
            dmma884(w[q - 1][u][0], w[q - 1][u][1], fDtA[1], c1[u]);
          }
        }
        if (q < nq1) {
          double dx[2][2], dy[2][2], dz[2][2];
#pragma unroll
          for (int u = 0; u < 2; ++u) {
            dx[u][0] = dx[u][1] = dy[u][0] = dy[u][1] = dz[u][0] = dz[u][1] = 0.0;
            dmma884(dx[u][0], dx[u][1], fDA[0], b0[u]);                // d_x u^ = sum_qa Dh[qa'][qa] u^[qa][qb]
            dmma884(dy[u][0], dy[u][1], uh[q][u][0], fDB[0]);          // d_y u^ = sum_qb u^[qa][qb] Dh[qb'][qb]
          }
#pragma unroll
          for (int u = 0; u < 2; ++u) {
            dmma884(dx[u][0], dx[u][1], fDA[1], b1[u]);
            dmma884(dy[u][0], dy[u][1], uh[q][u][1], fDB[1]);
          }
          {
            double dzo[2][2] = {{0.0, 0.0}, {0.0, 0.0}};               // d_z u^ in the lane's registers (even / odd partial sums)
#pragma unroll
            for (int r = 0; r < nq1; ++r) {
              const double dh = c_sf_dhat[P][q * 8 + r];
#pragma unroll
              for (int u = 0; u < 2; ++u) {
                if (r & 1) { dzo[u][0] = fma(dh, uh[r][u][0], dzo[u][0]); dzo[u][1] = fma(dh, uh[r][u][1], dzo[u][1]); }
                else { dz[u][0] = fma(dh, uh[r][u][0], dz[u][0]); dz[u][1] = fma(dh, uh[r][u][1], dz[u][1]); }
              }
            }
#pragma unroll
            for (int u = 0; u < 2; ++u) { dz[u][0] += dzo[u][0]; dz[u][1] += dzo[u][1]; }
          }
          const double2* cq = reinterpret_cast<const double2*>(coef_s) + (q * 7) * 32 + lane;
          const double2 W0 = cq[0], Gxx = cq[32], Gxy = cq[64], Gxz = cq[96], Gyy = cq[128], Gyz = cq[160], Gzz = cq[192];
          double gz[2][2];
#pragma unroll
          for (int u = 0; u < 2; ++u) {
            double gx0, gx1, gy0, gy1;
            gx0 = fma(Gxx.x, dx[u][0], fma(Gxy.x, dy[u][0], Gxz.x * dz[u][0]));
            gx1 = fma(Gxx.y, dx[u][1], fma(Gxy.y, dy[u][1], Gxz.y * dz[u][1]));
            gy0 = fma(Gxy.x, dx[u][0], fma(Gyy.x, dy[u][0], Gyz.x * dz[u][0]));
            gy1 = fma(Gxy.y, dx[u][1], fma(Gyy.y, dy[u][1], Gyz.y * dz[u][1]));
            gz[u][0] = fma(Gxz.x, dx[u][0], fma(Gyz.x, dy[u][0], Gzz.x * dz[u][0]));
            gz[u][1] = fma(Gxz.y, dx[u][1], fma(Gyz.y, dy[u][1], Gzz.y * dz[u][1]));
            w[q][u][0] = fma(W0.x, uh[q][u][0], w[q][u][0]);
            w[q][u][1] = fma(W0.y, uh[q][u][1], w[q][u][1]);
            dmma884(w[q][u][0], w[q][u][1], gy0, fDtB[0]);             // += sum_qb g_y[qa][qb] Dh[qb][qb'']
            dmma884(w[q][u][0], w[q][u][1], gy1, fDtB[1]);
            *reinterpret_cast<double2*>(scrB + u * kSfScrSlab + so_w) = make_double2(gx0, gx1);
          }
#pragma unroll
          for (int r = 0; r < nq1; ++r) {
            const double dh = c_sf_dhat[P][q * 8 + r];                 // += Dh[q][r] g_z[q]
#pragma unroll
            for (int u = 0; u < 2; ++u) {
              w[r][u][0] = fma(dh, gz[u][0], w[r][u][0]);
              w[r][u][1] = fma(dh, gz[u][1], w[r][u][1]);
            }
          }
        }
      }

      // ---- back to the nodes: y = (Phi x Phi x Phi)^T w; slabs alternate between the two scratch buffers ------------
      double z[n1][2][2];
#pragma unroll
      for (int c = 0; c < n1; ++c)
#pragma unroll
        for (int u = 0; u < 2; ++u) z[c][u][0] = z[c][u][1] = 0.0;
#pragma unroll
      for (int q = 0; q < nq1; ++q)
#pragma unroll
        for (int c = 0; c < n1; ++c) {
          const double ph = c_sf_phi[P][q * 8 + c];
#pragma unroll
          for (int u = 0; u < 2; ++u) {
            z[c][u][0] = fma(ph, w[q][u][0], z[c][u][0]);
            z[c][u][1] = fma(ph, w[q][u][1], z[c][u][1]);
          }
        }
#pragma unroll
      for (int c = 0; c < n1; ++c) {
        double* scr = (c & 1) ? scrB : scrA;
#pragma unroll
        for (int u = 0; u < 2; ++u) {
          double y0 = 0.0, y1 = 0.0;
          dmma884(y0, y1, z[c][u][0], fPhiTB[0]);                      // y1[c][b][qa] = sum_qb z[qa][qb] Phi[qb][b]
          dmma884(y0, y1, z[c][u][1], fPhiTB[1]);
          *reinterpret_cast<double2*>(scr + u * kSfScrSlab + so_w) = make_double2(y0, y1);
        }
        __syncwarp();
        double y[2][2];
#pragma unroll
        for (int u = 0; u < 2; ++u) {
          const double b0 = scr[u * kSfScrSlab + so_r0], b1 = scr[u * kSfScrSlab + so_r1];
          y[u][0] = y[u][1] = 0.0;
          dmma884(y[u][0], y[u][1], fPhiTA[0], b0);                    // y[c][b][a] = sum_qa Phi[qa][a] y1[c][b][qa]
          dmma884(y[u][0], y[u][1], fPhiTA[1], b1);
        }
        // lane (g, t): nodes (a = g, b = 2t + e, c); the result overwrites the two columns:  s_l y_l - c x_l [first]
#pragma unroll
        for (int e = 0; e < 2; ++e) {
          const int bi = 2 * t + e;
          if (g < n1 && bi < n1) {
            const int l = g + n1 * bi + nn * c;
            S* xp = reinterpret_cast<S*>(xt + sf_pair_off<S>(l, pp));
            const double2 tb = tab_s[l];
            const double2 xo = sf_ld_pair(xp);
            sf_st_pair(xp, fma(tb.x, y[0][e], -tb.y * xo.x), fma(tb.x, y[1][e], -tb.y * xo.y));
          }
        }
      }
      __syncwarp();                                                    // scratch free for the next pair of columns
    }
    __syncthreads();                                                   // the whole tile holds H~^loc X - c X [first]
    }
    // The tile coordinates are re-derived from the ticket in shared memory (a volatile read) instead of being kept in
    // registers across the column loop above, which needs every register it can get.
    {
    const long long ticket = *reinterpret_cast<volatile long long*>(&ticket_s[iter & 1]);
    int32_t* idx_s = idx_all + (iter & 1) * kIdxStride;
    int32_t* idx_n = idx_all + ((iter + 1) & 1) * kIdxStride;
    const int pos = (int)(ticket / nct), jt = (int)(ticket % nct);
    const int cell = pd.pos_cell[pos];
    const int col0 = jt * TN;
    const int ncols = min(TN, a.B - col0);
    const int64_t cp0 = sf.cell_proj_ptr[cell];
    const int np = (int)(sf.cell_proj_ptr[cell + 1] - cp0);
    const double alpha = a.alpha, beta = a.beta;
    const double* Ps = Ps_all + (iter & 1) * kSfMaxProj * TN;

    // ---- assembly + recurrence (steps 4-5) and the projector term C~^c P (Alg. 4 step 5) -------------------------
    // The coefficient fields are dead now: the projector columns of the cell, s_l C^c_{l,j} ([np][mpad] FP64, contiguous),
    // arrive in their place by one bulk copy while the dependency flags and the old target rows are fetched.
    const long long ticket_n = ticket_s[(iter + 1) & 1];
    const bool has_next = ticket_n < pd.n_tiles;
    int cell_n = 0, col0_n = 0;
    if (has_next) load_small(ticket_n, cell_n, col0_n);
    double* crow_s = coef_s;
    const int npc = min(np, kSfCrowChunk);
    if (tid == 0 && np > 0) {
      asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
      mbar_expect_tx(bar + 1, (uint32_t)(npc * mpad * sizeof(double)));
      bulk_g2s(crow_s, sf.crows + cp0 * mpad, (uint32_t)(npc * mpad * sizeof(double)), bar + 1);
    }
    if (!a.atomic) {
      const int d0 = pd.dep_ptr[pos], nd = pd.dep_ptr[pos + 1] - d0;
      for (int d = lane; d < nd; d += 32) {
        const uint32_t* f = pd.flags + (int64_t)pd.dep_pos[d0 + d] * nct + jt;
        while (ld_acquire_gpu(f) != pd.epoch) __nanosleep(64);
      }
      __syncwarp();
    }
    {
      // thread mapping = C fragment of an m8n8 tile: warp step = 8 rows (r = 8 mt + g) x TN columns, lane holds columns
      // 8 nt + 2t + {0, 1} of every 8-column block nt: one 16-byte (FP64) store per block, 64 contiguous bytes per 4 lanes
      constexpr int nmt = (mc + 7) / 8;
      constexpr int kSteps = (nmt + kSfWarps - 1) / kSfWarps;
      const bool use_t = (beta != 0.0) && !a.atomic;
      // old target rows of the first contributions (the -beta Y_{k-2} term), all in flight at once
      S told[kSteps][NT][2];
#pragma unroll
      for (int i = 0; i < kSteps; ++i) {
        const int r = 8 * (warp + i * kSfWarps) + g;
#pragma unroll
        for (int nt = 0; nt < NT; ++nt) told[i][nt][0] = told[i][nt][1] = (S)0;
        if (use_t && r < mc) {
          const int idx = idx_s[r];
          if (idx < 0) {
            const S* trow = a.Tg + (int64_t)(idx & 0x7fffffff) * a.ldt + col0 + 2 * t;
#pragma unroll
            for (int nt = 0; nt < NT; ++nt)
              if (8 * nt + 2 * t < ncols) {
                if constexpr (sizeof(S) == 8) {
                  const double2 u2 = ld_cg_d2(trow + 8 * nt);
                  told[i][nt][0] = u2.x; told[i][nt][1] = u2.y;
                } else {
                  float x, y;
                  asm volatile("ld.global.cg.v2.f32 {%0,%1}, [%2];" : "=f"(x), "=f"(y) : "l"(trow + 8 * nt) : "memory");
                  told[i][nt][0] = x; told[i][nt][1] = y;
                }
              }
          }
        }
      }
      // B fragments of the projector coefficients of the cell: P[j = 4s + t][column 8 nt + g]
      double pb[2][NT];
#pragma unroll
      for (int s = 0; s < 2; ++s)
#pragma unroll
        for (int nt = 0; nt < NT; ++nt) pb[s][nt] = Ps[(4 * s + t) * TN + 8 * nt + g];
      if (np > 0) { mbar_wait(bar + 1, phase_c); phase_c ^= 1u; }
#pragma unroll
      for (int i = 0; i < kSteps; ++i) {
        const int mt = warp + i * kSfWarps;
        if (mt >= nmt) break;
        const int r = 8 * mt + g;                           // < mpad: the padding rows of the tile exist (never stored)
        double v[NT][2];
#pragma unroll
        for (int nt = 0; nt < NT; ++nt) {
          const double2 x2 = sf_ld_pair(reinterpret_cast<const S*>(xt + sf_pair_off<S>(r, 4 * nt + t)));
          v[nt][0] = x2.x; v[nt][1] = x2.y;
        }
        if (np > 0) {
          const double a0 = (t < npc) ? crow_s[t * mpad + r] : 0.0;
          const double a1 = (4 + t < npc) ? crow_s[(4 + t) * mpad + r] : 0.0;
#pragma unroll
          for (int nt = 0; nt < NT; ++nt) {
            dmma884(v[nt][0], v[nt][1], a0, pb[0][nt]);     // += sum_j C~[r][j] P[j][col]
            dmma884(v[nt][0], v[nt][1], a1, pb[1][nt]);
          }
          for (int j0 = kSfCrowChunk; j0 < np; j0 += 8) {  // more projectors than one chunk: straight from global
            const int ja = j0 + t, jb = j0 + 4 + t;
            const double e0 = (ja < np) ? sf.crows[(cp0 + ja) * mpad + r] : 0.0;
            const double e1 = (jb < np) ? sf.crows[(cp0 + jb) * mpad + r] : 0.0;
#pragma unroll
            for (int nt = 0; nt < NT; ++nt) {
              dmma884(v[nt][0], v[nt][1], e0, ja < np ? Ps[ja * TN + 8 * nt + g] : 0.0);
              dmma884(v[nt][0], v[nt][1], e1, jb < np ? Ps[jb * TN + 8 * nt + g] : 0.0);
            }
          }
        }
        if (r >= mc) continue;
        const int idx = idx_s[r];
        S* trow = a.Tg + (int64_t)(idx & 0x7fffffff) * a.ldt + col0 + 2 * t;
        const bool add = a.atomic || idx >= 0;
#pragma unroll
        for (int nt = 0; nt < NT; ++nt) {
          if (8 * nt + 2 * t >= ncols) continue;
          if (add) {
            atomicAdd(trow + 8 * nt, (S)(alpha * v[nt][0]));
            atomicAdd(trow + 8 * nt + 1, (S)(alpha * v[nt][1]));
          } else {
            sf_st_pair(trow + 8 * nt, fma(alpha, v[nt][0], -beta * (double)told[i][nt][0]),
                       fma(alpha, v[nt][1], -beta * (double)told[i][nt][1]));
          }
        }
      }
    }
    phase ^= 1u;
    if (has_next) store_small(idx_n, Ps_all + ((iter + 1) & 1) * kSfMaxProj * TN);
    __threadfence();                                               // (before the copies are issued: the fence would wait for them)
    asm volatile("fence.proxy.async.shared::cta;" ::: "memory");   // generic accesses to the tile rows before the next TMA writes
    __syncthreads();                                               // tile assembled and fenced; next index list visible
    if (tid == 0 && !a.atomic) st_release_gpu(pd.flags + (int64_t)pos * nct + jt, pd.epoch);
    if (has_next && warp == 0) issue_tile(idx_n, cell_n, col0_n);
    }
  }
}
