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
// Mapping (one warp = one column at a time; lane = 4 g + t):
//   * a 1-D contraction over the index that is spread over t runs as two m8n8k4 DMMAs per 8 x 8 slab; chaining
//     "matrix x data" (data = B operand, read from shared memory) with "data x matrix" (data = A operand = the C
//     fragment of the previous product: with the contraction index ordered (2t, 2t+1) the C fragment IS the A fragment
//     pair) applies two directions without moving data; the third direction lives in the lane's registers and is plain
//     DFMA with the 1-D matrices as constant-bank operands; the x-direction of the gradient and of the final
//     interpolation needs the slab transposed, which is one trip through a per-warp scratch in shared memory.
//   * canonical register layout of a field on the Gauss grid: lane (g, t) holds (qa = g, qb = 2t + {0, 1}) for all qc.
//   * tile = (cell, 16 FP64 | 32 FP32 columns); its rows are gathered by TMA tile::gather4 with SWIZZLE_128B (row =
//     128 bytes), so that the B-fragment loads (32 lanes = 32 different rows, one column) spread over the banks; the
//     result of a column overwrites the column in place and the CTA then assembles the tile row by row (128-byte rows).
#pragma once

constexpr int kSfThreads = 128;
constexpr int kSfWarps = kSfThreads / 32;
constexpr int kSfScrPitch = 10;                  // doubles per row of a scratch slab (bank-conflict-free, 16-byte rows)
constexpr int kSfScrSlab = 8 * kSfScrPitch;
constexpr int kSfMaxProj = 32;                   // projectors touching one cell (more: the dense kernel takes the operator)
template <typename S> __host__ __device__ constexpr int sf_cpc() { return 16 / (int)sizeof(S); }        // columns per 16-byte chunk
template <typename S> __host__ __device__ constexpr int sf_tile_cols() { return 8 * sf_cpc<S>(); }      // 16 | 32

// 1-D tables of the degrees in use, zero-padded to 8 x 8: Phi[q][i] = l_i(x_q), Dh[q'][q] = (d/dx) lhat_q (x_q')
__constant__ double c_sf_phi[7][64];
__constant__ double c_sf_dhat[7][64];

struct SfDev {
  const double* __restrict__ coef;           // [n_cells][nq1][7][32 lanes][2]: W0, Gxx, Gxy, Gxz, Gyy, Gyz, Gzz at the lane's points
  const double* __restrict__ sloc;           // [n_cells][mpad]  M^-1/2 at the nodes of the cell
  const double* __restrict__ crows;          // [nnz_cell_proj][m_cell]  s_l C^c_{l,j}
  const int64_t* __restrict__ cell_proj_ptr; // [n_cells + 1]
  double cshift;                             // spectral shift c of the running filter (0 for apply_H)
};

template <int P, typename S>
size_t sf_smem_bytes(const Op* op) {
  constexpr int nq1 = P + 2;
  size_t b = 1024;                                                     // alignment slack of the swizzled tile
  b += (size_t)op->mpad * 128;                                         // tile rows
  b += (size_t)nq1 * 7 * 64 * sizeof(double);                          // coefficient fields of the cell
  b += (size_t)kSfWarps * 8 * kSfScrSlab * sizeof(double);             // per-warp transposition scratch
  b += (size_t)op->mpad * 16;                                          // {s_l, c or 0} per node
  b += (size_t)kSfMaxProj * sf_tile_cols<S>() * sizeof(double);        // rows of P for the cell
  b += (size_t)(op->mpad + kSfMaxProj) * sizeof(int32_t) + 64;         // index list, barrier, tickets
  return b;
}

template <typename S>
__device__ __forceinline__ uint32_t sf_xoff(int l, int j) {          // byte offset of (row l, column j) in the swizzled tile
  constexpr int cpc = sf_cpc<S>();
  return (uint32_t)l * 128u + ((uint32_t)((j / cpc) ^ (l & 7)) << 4) + (uint32_t)(j % cpc) * (uint32_t)sizeof(S);
}

template <int P, typename S>
__global__ void __launch_bounds__(kSfThreads, 2) k_apply_sf(ApplyDev<S> a, SfDev sf, PersistDev pd,
                                                            const __grid_constant__ CUtensorMap tmX) {
  constexpr int n1 = P + 1, nq1 = P + 2, nn = n1 * n1, mc = n1 * nn;
  constexpr int TN = sf_tile_cols<S>(), CPC = sf_cpc<S>();
  constexpr int coef_elems = nq1 * 7 * 64;
  extern __shared__ unsigned char smem_dyn[];
  unsigned char* base = reinterpret_cast<unsigned char*>(((uintptr_t)smem_dyn + 1023) & ~(uintptr_t)1023);
  const int mpad = a.mpad;
  unsigned char* xt = base;                                                         // [mpad][128 B], swizzled
  double* coef_s = reinterpret_cast<double*>(xt + (size_t)mpad * 128);              // [nq1][7][32][2]
  double* scr_all = coef_s + coef_elems;                                            // [warps][8][kSfScrSlab]
  double2* tab_s = reinterpret_cast<double2*>(scr_all + kSfWarps * 8 * kSfScrSlab); // [mpad]
  double* Ps = reinterpret_cast<double*>(tab_s + mpad);                             // [kSfMaxProj][TN]
  uint64_t* bar = reinterpret_cast<uint64_t*>(Ps + kSfMaxProj * TN);
  long long* ticket_s = reinterpret_cast<long long*>(bar + 1);                      // [2]
  int32_t* idx_s = reinterpret_cast<int32_t*>(ticket_s + 2);                        // [mpad + kSfMaxProj]

  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  const int g = lane >> 2, t = lane & 3;
  const int nct = a.n_col_tiles;
  const double alpha = a.alpha, beta = a.beta;
  double* scr = scr_all + warp * 8 * kSfScrSlab;

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
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    ticket_s[0] = (long long)(atomicAdd(pd.counter, 1ull) - pd.ticket_base);
  }
  __syncthreads();

  uint32_t phase = 0;
  for (int iter = 0;; ++iter) {
    const long long ticket = ticket_s[iter & 1];
    if (ticket >= pd.n_tiles) break;
    const int pos = (int)(ticket / nct), jt = (int)(ticket % nct);
    const int cell = pd.pos_cell[pos];
    const int col0 = jt * TN;
    const int ncols = min(TN, a.B - col0);
    const int32_t* gi = a.gidx + a.idx_off[cell];
    const int64_t cp0 = sf.cell_proj_ptr[cell];
    const int np = (int)(sf.cell_proj_ptr[cell + 1] - cp0);
    if (tid == 0) ticket_s[(iter + 1) & 1] = (long long)(atomicAdd(pd.counter, 1ull) - pd.ticket_base);
    for (int k = tid; k < mpad + np; k += kSfThreads) {
      const int idx = gi[k];
      idx_s[k] = idx;
      if (k < mpad) tab_s[k] = make_double2(k < mc ? sf.sloc[(int64_t)cell * mpad + k] : 0.0, (idx < 0) ? sf.cshift : 0.0);
    }
    for (int e = tid; e < np * TN; e += kSfThreads) {
      const int jj = e / TN, cc = e % TN;
      Ps[e] = (cc < ncols) ? (double)a.P[(int64_t)gi[mpad + jj] * a.ldp + col0 + cc] : 0.0;
    }
    __syncthreads();   // idx_s / tab_s / Ps visible; every thread is done with the previous tile's rows (its epilogue)
    if (warp == 0) {
      if (lane == 0) {
        mbar_expect_tx(bar, (uint32_t)mpad * 128u + (uint32_t)(coef_elems * sizeof(double)));
        bulk_g2s(coef_s, sf.coef + (int64_t)cell * coef_elems, (uint32_t)(coef_elems * sizeof(double)), bar);
      }
      __syncwarp();
      for (int r4 = lane; r4 < mpad / 4; r4 += 32)
        tma_gather4(xt + (size_t)r4 * 512, &tmX, col0, idx_s[4 * r4] & 0x7fffffff, idx_s[4 * r4 + 1] & 0x7fffffff,
                    idx_s[4 * r4 + 2] & 0x7fffffff, idx_s[4 * r4 + 3] & 0x7fffffff, bar);
    }
    mbar_wait(bar, phase);
    phase ^= 1u;

    // ------------------------------------------------------------------------------------------------------------
    // one column at a time per warp
    // ------------------------------------------------------------------------------------------------------------
    for (int j = warp; j < ncols; j += kSfWarps) {
      // ---- forward interpolation: u^ = (Phi x Phi x Phi) u ----------------------------------------------------
      double T2[n1][2];
      {
        double d[n1][2];
#pragma unroll
        for (int s = 0; s < 2; ++s) {
          double bv[n1];
          const int ai = 4 * s + t;
          const bool ok = (ai < n1) && (g < n1);
#pragma unroll
          for (int c = 0; c < n1; ++c) {
            const int l = ai + n1 * g + nn * c;
            bv[c] = 0.0;
            if (ok) bv[c] = (double)(*reinterpret_cast<const S*>(xt + sf_xoff<S>(l, j))) * tab_s[l].x;
          }
#pragma unroll
          for (int c = 0; c < n1; ++c) {
            if (s == 0) d[c][0] = d[c][1] = 0.0;
            dmma884(d[c][0], d[c][1], fPhiA[s], bv[c]);               // T1[c][b][qa] = sum_a Phi[qa][a] u[c][b][a]
          }
        }
#pragma unroll
        for (int c = 0; c < n1; ++c) T2[c][0] = T2[c][1] = 0.0;
#pragma unroll
        for (int s = 0; s < 2; ++s)
#pragma unroll
          for (int c = 0; c < n1; ++c) dmma884(T2[c][0], T2[c][1], d[c][s], fPhiB[s]);   // T2[c][qb][qa] = sum_b T1 Phi[qb][b]
      }
      double uh[nq1][2], w[nq1][2];
#pragma unroll
      for (int q = 0; q < nq1; ++q) {
        double s0 = 0.0, s1 = 0.0;
#pragma unroll
        for (int c = 0; c < n1; ++c) {
          s0 = fma(c_sf_phi[P][q * 8 + c], T2[c][0], s0);
          s1 = fma(c_sf_phi[P][q * 8 + c], T2[c][1], s1);
        }
        uh[q][0] = s0; uh[q][1] = s1;
        w[q][0] = w[q][1] = 0.0;
      }
      // slabs of u^ to the scratch (for the x-derivative the slab is read back with qa as the contraction index)
#pragma unroll
      for (int q = 0; q < nq1; ++q)
        *reinterpret_cast<double2*>(scr + q * kSfScrSlab + g * kSfScrPitch + 2 * t) = make_double2(uh[q][0], uh[q][1]);
      __syncwarp();

      // ---- Gauss grid: gradient, metric / potential, transposed gradient ---------------------------------------
#pragma unroll
      for (int q = 0; q < nq1; ++q) {
        double dx[2] = {0.0, 0.0}, dy[2] = {0.0, 0.0}, dz[2] = {0.0, 0.0};
        const double b0 = scr[q * kSfScrSlab + t * kSfScrPitch + g];
        const double b1 = scr[q * kSfScrSlab + (4 + t) * kSfScrPitch + g];
        dmma884(dx[0], dx[1], fDA[0], b0);                             // d_x u^ = sum_qa Dh[qa'][qa] u^[qa][qb]
        dmma884(dx[0], dx[1], fDA[1], b1);
        dmma884(dy[0], dy[1], uh[q][0], fDB[0]);                       // d_y u^ = sum_qb u^[qa][qb] Dh[qb'][qb]
        dmma884(dy[0], dy[1], uh[q][1], fDB[1]);
#pragma unroll
        for (int r = 0; r < nq1; ++r) {
          dz[0] = fma(c_sf_dhat[P][q * 8 + r], uh[r][0], dz[0]);      // d_z u^ in the lane's registers
          dz[1] = fma(c_sf_dhat[P][q * 8 + r], uh[r][1], dz[1]);
        }
        const double2* cq = reinterpret_cast<const double2*>(coef_s) + (q * 7) * 32 + lane;
        const double2 W0 = cq[0], Gxx = cq[32], Gxy = cq[64], Gxz = cq[96], Gyy = cq[128], Gyz = cq[160], Gzz = cq[192];
        double gx[2], gy[2], gz[2];
        gx[0] = fma(Gxx.x, dx[0], fma(Gxy.x, dy[0], Gxz.x * dz[0]));
        gx[1] = fma(Gxx.y, dx[1], fma(Gxy.y, dy[1], Gxz.y * dz[1]));
        gy[0] = fma(Gxy.x, dx[0], fma(Gyy.x, dy[0], Gyz.x * dz[0]));
        gy[1] = fma(Gxy.y, dx[1], fma(Gyy.y, dy[1], Gyz.y * dz[1]));
        gz[0] = fma(Gxz.x, dx[0], fma(Gyz.x, dy[0], Gzz.x * dz[0]));
        gz[1] = fma(Gxz.y, dx[1], fma(Gyz.y, dy[1], Gzz.y * dz[1]));
        w[q][0] = fma(W0.x, uh[q][0], w[q][0]);
        w[q][1] = fma(W0.y, uh[q][1], w[q][1]);
        dmma884(w[q][0], w[q][1], gy[0], fDtB[0]);                     // += sum_qb g_y[qa][qb] Dh[qb][qb'']
        dmma884(w[q][0], w[q][1], gy[1], fDtB[1]);
#pragma unroll
        for (int r = 0; r < nq1; ++r) {
          w[r][0] = fma(c_sf_dhat[P][q * 8 + r], gz[0], w[r][0]);     // += Dh[q][r] g_z[q]
          w[r][1] = fma(c_sf_dhat[P][q * 8 + r], gz[1], w[r][1]);
        }
        __syncwarp();                                                  // every lane has read slab q of u^
        *reinterpret_cast<double2*>(scr + q * kSfScrSlab + g * kSfScrPitch + 2 * t) = make_double2(gx[0], gx[1]);
      }
      __syncwarp();
#pragma unroll
      for (int q = 0; q < nq1; ++q) {
        const double b0 = scr[q * kSfScrSlab + t * kSfScrPitch + g];
        const double b1 = scr[q * kSfScrSlab + (4 + t) * kSfScrPitch + g];
        dmma884(w[q][0], w[q][1], fDtA[0], b0);                        // += sum_qa Dh[qa][qa''] g_x[qa][qb]
        dmma884(w[q][0], w[q][1], fDtA[1], b1);
      }
      __syncwarp();                                                    // slabs of g_x consumed

      // ---- back to the nodes: y = (Phi x Phi x Phi)^T w -----------------------------------------------------------
#pragma unroll
      for (int c = 0; c < n1; ++c) {
        double z0 = 0.0, z1 = 0.0;
#pragma unroll
        for (int q = 0; q < nq1; ++q) {
          z0 = fma(c_sf_phi[P][q * 8 + c], w[q][0], z0);
          z1 = fma(c_sf_phi[P][q * 8 + c], w[q][1], z1);
        }
        double y0 = 0.0, y1 = 0.0;
        dmma884(y0, y1, z0, fPhiTB[0]);                                // y1[c][b][qa] = sum_qb z[qa][qb] Phi[qb][b]
        dmma884(y0, y1, z1, fPhiTB[1]);
        *reinterpret_cast<double2*>(scr + c * kSfScrSlab + g * kSfScrPitch + 2 * t) = make_double2(y0, y1);
      }
      __syncwarp();
#pragma unroll
      for (int c = 0; c < n1; ++c) {
        const double b0 = scr[c * kSfScrSlab + t * kSfScrPitch + g];
        const double b1 = scr[c * kSfScrSlab + (4 + t) * kSfScrPitch + g];
        double y[2] = {0.0, 0.0};
        dmma884(y[0], y[1], fPhiTA[0], b0);                            // y[c][b][a] = sum_qa Phi[qa][a] y1[c][b][qa]
        dmma884(y[0], y[1], fPhiTA[1], b1);
        // lane (g, t): nodes (a = g, b = 2t + e, c); result of the column overwrites the column:  s_l y_l - c x_l [first]
#pragma unroll
        for (int e = 0; e < 2; ++e) {
          const int bi = 2 * t + e;
          if (g < n1 && bi < n1) {
            const int l = g + n1 * bi + nn * c;
            S* xp = reinterpret_cast<S*>(xt + sf_xoff<S>(l, j));
            const double2 tb = tab_s[l];
            *xp = (S)fma(tb.x, y[e], -tb.y * (double)(*xp));
          }
        }
      }
      __syncwarp();                                                    // scratch free for the next column
    }
    __syncthreads();                                                   // the whole tile holds H~^loc X - c X [first]

    // ---- assembly + recurrence (steps 4-5) and the projector term C~^c P (Alg. 4 step 5) -------------------------
    if (!a.atomic) {
      const int d0 = pd.dep_ptr[pos], nd = pd.dep_ptr[pos + 1] - d0;
      for (int d = lane; d < nd; d += 32) {
        const uint32_t* f = pd.flags + (int64_t)pd.dep_pos[d0 + d] * nct + jt;
        while (ld_acquire_gpu(f) != pd.epoch) __nanosleep(64);
      }
      __syncwarp();
    }
    {
      const int rsub = tid >> 3, ch = tid & 7;
      const bool colok = ch * CPC < ncols;
      for (int r = rsub; r < mc; r += kSfThreads / 8) {
        double v[CPC];
        if constexpr (sizeof(S) == 8) {
          const double2 u = *reinterpret_cast<const double2*>(xt + (size_t)r * 128 + ((ch ^ (r & 7)) << 4));
          v[0] = u.x; v[1] = u.y;
        } else {
          const float4 u = *reinterpret_cast<const float4*>(xt + (size_t)r * 128 + ((ch ^ (r & 7)) << 4));
          v[0] = u.x; v[1] = u.y; v[2] = u.z; v[3] = u.w;
        }
        for (int jj = 0; jj < np; ++jj) {
          const double cj = sf.crows[(cp0 + jj) * mc + r];
#pragma unroll
          for (int k = 0; k < CPC; ++k) v[k] = fma(cj, Ps[jj * TN + ch * CPC + k], v[k]);
        }
        if (!colok) continue;
        const int idx = idx_s[r];
        S* trow = a.Tg + (int64_t)(idx & 0x7fffffff) * a.ldt + col0 + ch * CPC;
        if (a.atomic || idx >= 0) {
#pragma unroll
          for (int k = 0; k < CPC; ++k) atomicAdd(trow + k, (S)(alpha * v[k]));
        } else {
          if (beta != 0.0) {
            if constexpr (sizeof(S) == 8) {
              const double2 u = ld_cg_d2(trow);
              v[0] = fma(alpha, v[0], -beta * u.x); v[1] = fma(alpha, v[1], -beta * u.y);
            } else {
              float4 u;
              asm volatile("ld.global.cg.v4.f32 {%0,%1,%2,%3}, [%4];" : "=f"(u.x), "=f"(u.y), "=f"(u.z), "=f"(u.w) : "l"(trow) : "memory");
              v[0] = fma(alpha, v[0], -beta * (double)u.x); v[1] = fma(alpha, v[1], -beta * (double)u.y);
              v[2] = fma(alpha, v[2], -beta * (double)u.z); v[3] = fma(alpha, v[3], -beta * (double)u.w);
            }
          } else {
#pragma unroll
            for (int k = 0; k < CPC; ++k) v[k] *= alpha;
          }
          if constexpr (sizeof(S) == 8) *reinterpret_cast<double2*>(trow) = make_double2(v[0], v[1]);
          else *reinterpret_cast<float4*>(trow) = make_float4((float)v[0], (float)v[1], (float)v[2], (float)v[3]);
        }
      }
    }
    __threadfence();
    asm volatile("fence.proxy.async.shared::cta;" ::: "memory");   // generic accesses to the tile rows before the next TMA writes
    __syncthreads();
    if (tid == 0 && !a.atomic) st_release_gpu(pd.flags + (int64_t)pos * nct + jt, pd.epoch);
  }
}
