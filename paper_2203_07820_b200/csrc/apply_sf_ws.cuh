// Warp-specialised form of the sum-factorised fused H~ application + recurrence update (apply_sf.cuh), FE degree p <= 6.
// Included by apply_kernels.cu after apply_sf.cuh (same arithmetic, same data, same ticket / completion-flag protocol).
//
// Why: in k_apply_sf a CTA alternates between the column loop (the 1-D contractions, all FP64-pipe work) and the tile
// hand-over (dependency flags, old target rows, projector term, scatter, fence, index list and gather of the next tile).
// ncu (profiles/r02_sf_kernel.md) shows ~40 % of the warp samples in the hand-over or waiting for the next gather, and the
// FP64 pipe idles meanwhile.  Here ONE CTA per SM runs three roles on a ring of two tile buffers:
//   * 8 compute warps (two warpgroups, registers raised by setmaxnreg): column loop only.  A warp takes the column pairs
//     pp = warp, warp + 8, ... of tile j in buffer j & 1, overwrites them in place, arrives on done[j & 1] and goes on to
//     tile j + 1 in the other buffer: no CTA barrier, no global-memory access besides spills.
//   * 1 producer warp: draws the tickets; for tile j it fetches the index list and M^-1/2 of the cell (two bulk copies,
//     one tile ahead), waits until buffer j & 1 has been assembled, and issues the TMA row gather of X, the bulk copies
//     of the cell's quadrature fields and projector columns and the row gather of its P rows -- all onto full[j & 1].
//   * 3 assembler warps: for tile j they wait for done[j & 1] and for the completion flags of the cells that come
//     earlier in colour order, add the projector term C~^c P (Alg. 4 step 5: one k = 8 DMMA per 8 x 8 block), scale by
//     alpha and scatter the tile (store / red.add), release the tile's flag and hand the buffer back to the producer.
// So the hand-over of tile j and the gather of tile j + 2 run under the column loop of tile j + 1.
//
// Recurrence: the assembly has NO load from the target block.  The kernel computes either
//     T  = alpha (H~ - c) X        first contributions are stores (apply_H, first filter degree), or
//     T += alpha (H~ - c) X        every contribution is a red.add (accumulate = 1),
// and the filter loop (api.cu) runs the three-term recurrence in scaled blocks W_k = s_k Y_k with s_k = -s_{k-2} / beta_k,
// for which  Y_k = alpha_k (H~ - c) Y_{k-1} - beta_k Y_{k-2}  becomes  W_k = W_{k-2} + (s_k alpha_k / s_{k-1}) (H~ - c) W_{k-1}:
// the target block already holds the additive term (|s_k| = T_k(t0) / T_{k mod 2}(t0): the unnormalised polynomials).
//
// Shared memory (p = 6, bytes): 2 x 44,032 tile rows + 2 x 28,672 fields + 2 x 22,016 projector columns + 2 x 2,048 P rows
// + 3 x 4,192 index list / M^-1/2 + 8 x 2,560 scratch ~ 221 KB.
#pragma once

constexpr int kWsComputeWarps = 8;
constexpr int kWsHelperWarps = 4;                 // warp 8: producer; warps 9-11: assemblers
constexpr int kWsAsmWarps = kWsHelperWarps - 1;
constexpr int kWsThreads = 32 * (kWsComputeWarps + kWsHelperWarps);
// registers after setmaxnreg: 256 x 216 + 128 x 72 = 256 x 232 + 128 x 40 = 64,512 = 384 x 168 (the launch allocation).
// FP64 tiles (one column pair per compute warp) need the faster assembler: at 72 registers its two m-tiles in flight are
// spill-free and the column loop still is at 216 (measured: 224 / 56 -> 216 / 72 +2 % at config 5, 208 / 88 no further gain);
// FP32 tiles (two pairs per warp) leave the assembler slack.
template <typename S> __host__ __device__ constexpr int ws_regs_compute() { return sizeof(S) == 8 ? 216 : 232; }
template <typename S> __host__ __device__ constexpr int ws_regs_helper() { return sizeof(S) == 8 ? 72 : 40; }

// KP = k-point variant: a column pair is one complex column (re, im); ten fields per Gauss point (the last three carry
// w detJ J^-1 k); no projector data here -- the back-projection C (D P) is k_proj_back's.
template <int P, typename S, bool KP = false>
struct WsSmem {
  static constexpr int n1 = P + 1, nq1 = P + 2, mc = n1 * n1 * n1, mpad = (mc + 7) / 8 * 8;
  static constexpr int TN = sf_tile_cols<S>();
  static constexpr int tile_bytes = (mpad * 128 + 1023) / 1024 * 1024;      // TMA swizzle atoms: 1024-byte aligned buffers
  static constexpr int NF = KP ? 10 : 7;                                    // fields per Gauss point
  static constexpr int coef_elems = nq1 * NF * 64;
  static constexpr int coef_bytes = coef_elems * 8;
  static constexpr int crow_bytes = KP ? 0 : (kSfCrowChunk * mpad * 8 + 127) / 128 * 128;
  static constexpr int ps_bytes = KP ? 0 : kSfMaxProj * 128;                         // [kSfMaxProj][TN] of S: 128-byte rows
  static constexpr int idx_stride = mpad + kSfMaxProj;
  static constexpr int small_bytes = (idx_stride * 4 + mpad * 8 + 127) / 128 * 128;   // index list, then M^-1/2 (doubles)
  static constexpr int off_xt = 0;                                          // [2][tile_bytes]
  static constexpr int off_coef = off_xt + 2 * tile_bytes;                  // [2][coef_bytes]
  static constexpr int off_crow = off_coef + 2 * coef_bytes;                // [2][crow_bytes]
  static constexpr int off_ps = off_crow + 2 * crow_bytes;                  // [2][ps_bytes]
  static constexpr int off_small = off_ps + 2 * ps_bytes;                   // [3][small_bytes]
  static constexpr int off_scr = off_small + 3 * small_bytes;               // [8 warps][4][kSfScrSlab] doubles
  static constexpr int off_bar = off_scr + kWsComputeWarps * 4 * kSfScrSlab * 8;   // full[2], done[2], free[2], small[3], crow2
  static constexpr int off_ticket = off_bar + 10 * 8;                        // [4] long long
  static constexpr int off_frag = (off_ticket + 4 * 8 + 15) / 16 * 16;      // [16][32] doubles: per-lane fragments of the 1-D matrices
  static constexpr int bytes = off_frag + 16 * 32 * 8;
  static_assert(idx_stride * 4 % 16 == 0, "M^-1/2 follows the index list 16-byte aligned");
};

__device__ __forceinline__ void ws_asm_sync() { asm volatile("bar.sync 1, %0;" ::"n"(32 * kWsAsmWarps) : "memory"); }

template <int P, typename S, bool KP>
__global__ void __launch_bounds__(kWsThreads, 1) k_apply_sf_ws(ApplyDev<S> a, SfDev sf, PersistDev pd,
                                                               const __grid_constant__ CUtensorMap tmX,
                                                               const __grid_constant__ CUtensorMap tmP) {
  using L = WsSmem<P, S, KP>;
  constexpr int NF = L::NF;
  constexpr int n1 = L::n1, nq1 = L::nq1, nn = n1 * n1, mc = L::mc, mpad = L::mpad;
  constexpr int TN = L::TN;
  constexpr int NT = TN / 8;
  extern __shared__ __align__(1024) unsigned char smem_dyn[];
  uint64_t* bar_full = reinterpret_cast<uint64_t*>(smem_dyn + L::off_bar);      // [2] rows, fields, projector data landed
  uint64_t* bar_done = bar_full + 2;                                            // [2] column loop of the tile finished
  uint64_t* bar_free = bar_full + 4;                                            // [2] tile assembled: buffer free again
  uint64_t* bar_small = bar_full + 6;                                           // [3] index list + M^-1/2 landed
  uint64_t* bar_crow2 = bar_full + 9;                                           // projector columns 8.. of the cell landed
  volatile long long* ticket_s = reinterpret_cast<volatile long long*>(smem_dyn + L::off_ticket);   // [4] ring
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  const int g = lane >> 2, t = lane & 3;
  const int nct = a.n_col_tiles;
  const long long n_tiles = pd.n_tiles;

  if (tid == 0) {
    for (int b = 0; b < 2; ++b) {
      mbar_init(bar_full + b, 1);
      mbar_init(bar_done + b, kWsComputeWarps);
      mbar_init(bar_free + b, 1);
    }
    for (int s = 0; s < 3; ++s) mbar_init(bar_small + s, 1);
    mbar_init(bar_crow2, 1);
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
  }
  __syncthreads();

  if (warp < kWsComputeWarps) {
    // =============================================================================================================
    // compute warps: the column loop of apply_sf.cuh on tile j in buffer j & 1
    // =============================================================================================================
    asm volatile("setmaxnreg.inc.sync.aligned.u32 %0;" ::"n"(ws_regs_compute<S>()));
    double* scrA = reinterpret_cast<double*>(smem_dyn + L::off_scr) + warp * 4 * kSfScrSlab;
    double* scrB = scrA + 2 * kSfScrSlab;
    const int so_w = g * kSfScrPitch + 2 * t;
    const int so_r0 = t * kSfScrPitch + g, so_r1 = (4 + t) * kSfScrPitch + g;
    // constant fragments of the 1-D matrices (k-step s: contraction index 4s + t for "matrix x data", 2t + s for "data x
    // matrix"), one 4 KB table in shared memory for all warps: sixteen doubles per lane that would otherwise be spilled
    // and come back from L2 at the start of every column pair
    double* frag_s = reinterpret_cast<double*>(smem_dyn + L::off_frag);
    if (warp == 0) {
#pragma unroll
      for (int s = 0; s < 2; ++s) {
        frag_s[(0 + s) * 32 + lane] = c_sf_phi[P][g * 8 + 4 * s + t];           // PhiA:  Phi[qa = g][a = 4s + t]
        frag_s[(2 + s) * 32 + lane] = c_sf_phi[P][g * 8 + 2 * t + s];           // PhiB:  Phi[qb = g][b = 2t + s]
        frag_s[(4 + s) * 32 + lane] = c_sf_dhat[P][g * 8 + 4 * s + t];          // DA:    Dh[qa' = g][qa = 4s + t]
        frag_s[(6 + s) * 32 + lane] = c_sf_dhat[P][g * 8 + 2 * t + s];          // DB:    Dh[qb' = g][qb = 2t + s]
        frag_s[(8 + s) * 32 + lane] = c_sf_dhat[P][(4 * s + t) * 8 + g];        // DtA:   Dh[qa = 4s + t][qa'' = g]
        frag_s[(10 + s) * 32 + lane] = c_sf_dhat[P][(2 * t + s) * 8 + g];       // DtB:   Dh[qb = 2t + s][qb'' = g]
        frag_s[(12 + s) * 32 + lane] = c_sf_phi[P][(4 * s + t) * 8 + g];        // PhiTA: Phi[qa = 4s + t][a = g]
        frag_s[(14 + s) * 32 + lane] = c_sf_phi[P][(2 * t + s) * 8 + g];        // PhiTB: Phi[qb = 2t + s][b = g]
      }
    }
    asm volatile("bar.sync 2, %0;" ::"n"(32 * kWsComputeWarps) : "memory");
    const double* fr = frag_s + lane;
#define fPhiA(s) fr[(0 + (s)) * 32]
#define fPhiB(s) fr[(2 + (s)) * 32]
#define fDA(s) fr[(4 + (s)) * 32]
#define fDB(s) fr[(6 + (s)) * 32]
#define fDtA(s) fr[(8 + (s)) * 32]
#define fDtB(s) fr[(10 + (s)) * 32]
#define fPhiTA(s) fr[(12 + (s)) * 32]
#define fPhiTB(s) fr[(14 + (s)) * 32]
    const double cshift = sf.cshift;
    // a run-time zero in the index of the 1-D tables: with compile-time addresses ptxas hoists a few dozen table entries
    // into registers for the whole kernel and spills them; this way every use is a uniform constant load next to its DFMAs
    const int zo = sf.zero;
    int set = 0;                                                      // j % 3
    for (int iter = 0;; ++iter) {
      const int b = iter & 1;
      mbar_wait(bar_full + b, (uint32_t)(iter >> 1) & 1u);
      const long long ticket = ticket_s[iter & 3];
      if (ticket >= n_tiles) break;
      mbar_wait(bar_small + set, (uint32_t)(iter / 3) & 1u);          // completed long ago: observed for the memory model only
      const int ncols = min(TN, a.B - (int)(ticket % nct) * TN);
      unsigned char* xt = smem_dyn + L::off_xt + b * L::tile_bytes;
      const double* coef_s = reinterpret_cast<const double*>(smem_dyn + L::off_coef + b * L::coef_bytes);
      const int32_t* idx_s = reinterpret_cast<const int32_t*>(smem_dyn + L::off_small + set * L::small_bytes);
      const double* sl_s = reinterpret_cast<const double*>(idx_s + L::idx_stride);

      for (int pp = warp; 2 * pp < ncols; pp += kWsComputeWarps) {
        double uh[nq1][2][2], w[nq1][2][2];
        {
          // ---- forward interpolation: u^ = (Phi x Phi x Phi) u --------------------------------------------------
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
                  const double sl = sl_s[l];
                  bv[c][0] = x2.x * sl; bv[c][1] = x2.y * sl;
                }
              }
#pragma unroll
              for (int c = 0; c < n1; ++c)
#pragma unroll
                for (int u = 0; u < 2; ++u) {
                  if (s == 0) d[c][u][0] = d[c][u][1] = 0.0;
                  dmma884(d[c][u][0], d[c][u][1], fPhiA(s), bv[c][u]);
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
                for (int u = 0; u < 2; ++u) dmma884(T2[c][u][0], T2[c][u][1], d[c][u][s], fPhiB(s));
          }
#pragma unroll
          for (int q = 0; q < nq1; ++q)
#pragma unroll
            for (int u = 0; u < 2; ++u) uh[q][u][0] = uh[q][u][1] = w[q][u][0] = w[q][u][1] = 0.0;
#pragma unroll
          for (int c = 0; c < n1; ++c)
#pragma unroll
            for (int q = 0; q < nq1; ++q) {
              const double ph = c_sf_phi[P][q * 8 + c + zo];
#pragma unroll
              for (int u = 0; u < 2; ++u) {
                uh[q][u][0] = fma(ph, T2[c][u][0], uh[q][u][0]);
                uh[q][u][1] = fma(ph, T2[c][u][1], uh[q][u][1]);
              }
            }
        }

        // ---- Gauss grid, slab by slab: gradient, metric / potential, transposed gradient ---------------------------
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
          __syncwarp();
          if (q > 0) {
#pragma unroll
            for (int u = 0; u < 2; ++u) {
              dmma884(w[q - 1][u][0], w[q - 1][u][1], fDtA(0), c0[u]);
              dmma884(w[q - 1][u][0], w[q - 1][u][1], fDtA(1), c1[u]);
            }
          }
          if (q < nq1) {
            double dx[2][2], dy[2][2], dz[2][2];
#pragma unroll
            for (int u = 0; u < 2; ++u) {
              dx[u][0] = dx[u][1] = dy[u][0] = dy[u][1] = dz[u][0] = dz[u][1] = 0.0;
              dmma884(dx[u][0], dx[u][1], fDA(0), b0[u]);
              dmma884(dy[u][0], dy[u][1], uh[q][u][0], fDB(0));
            }
#pragma unroll
            for (int u = 0; u < 2; ++u) {
              dmma884(dx[u][0], dx[u][1], fDA(1), b1[u]);
              dmma884(dy[u][0], dy[u][1], uh[q][u][1], fDB(1));
            }
            {
              double dzo[2][2] = {{0.0, 0.0}, {0.0, 0.0}};
#pragma unroll
              for (int r = 0; r < nq1; ++r) {
                const double dh = c_sf_dhat[P][q * 8 + r + zo];
#pragma unroll
                for (int u = 0; u < 2; ++u) {
                  if (r & 1) { dzo[u][0] = fma(dh, uh[r][u][0], dzo[u][0]); dzo[u][1] = fma(dh, uh[r][u][1], dzo[u][1]); }
                  else { dz[u][0] = fma(dh, uh[r][u][0], dz[u][0]); dz[u][1] = fma(dh, uh[r][u][1], dz[u][1]); }
                }
              }
#pragma unroll
              for (int u = 0; u < 2; ++u) { dz[u][0] += dzo[u][0]; dz[u][1] += dzo[u][1]; }
            }
            const double2* cq = reinterpret_cast<const double2*>(coef_s) + (q * NF) * 32 + lane;
            const double2 W0 = cq[0], Gxx = cq[32], Gxy = cq[64], Gxz = cq[96], Gyy = cq[128], Gyz = cq[160], Gzz = cq[192];
            if (KP) {
              // -i int N_j k.grad u (Eq. 30 last term) on (re, im) = (u = 0, u = 1):  re += kap.grad u_im,
              // im -= kap.grad u_re  with kap = w detJ J^-1 k
              const double2 Kx = cq[224], Ky = cq[256], Kz = cq[288];
              const double r0 = fma(Kx.x, dx[0][0], fma(Ky.x, dy[0][0], Kz.x * dz[0][0]));
              const double r1 = fma(Kx.y, dx[0][1], fma(Ky.y, dy[0][1], Kz.y * dz[0][1]));
              const double i0 = fma(Kx.x, dx[1][0], fma(Ky.x, dy[1][0], Kz.x * dz[1][0]));
              const double i1 = fma(Kx.y, dx[1][1], fma(Ky.y, dy[1][1], Kz.y * dz[1][1]));
              w[q][0][0] += i0; w[q][0][1] += i1;
              w[q][1][0] -= r0; w[q][1][1] -= r1;
            }
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
              dmma884(w[q][u][0], w[q][u][1], gy0, fDtB(0));
              dmma884(w[q][u][0], w[q][u][1], gy1, fDtB(1));
              *reinterpret_cast<double2*>(scrB + u * kSfScrSlab + so_w) = make_double2(gx0, gx1);
            }
#pragma unroll
            for (int r = 0; r < nq1; ++r) {
              const double dh = c_sf_dhat[P][q * 8 + r + zo];
#pragma unroll
              for (int u = 0; u < 2; ++u) {
                w[r][u][0] = fma(dh, gz[u][0], w[r][u][0]);
                w[r][u][1] = fma(dh, gz[u][1], w[r][u][1]);
              }
            }
          }
        }

        // ---- back to the nodes: y = (Phi x Phi x Phi)^T w ----------------------------------------------------------
        double z[n1][2][2];
#pragma unroll
        for (int c = 0; c < n1; ++c)
#pragma unroll
          for (int u = 0; u < 2; ++u) z[c][u][0] = z[c][u][1] = 0.0;
#pragma unroll
        for (int q = 0; q < nq1; ++q)
#pragma unroll
          for (int c = 0; c < n1; ++c) {
            const double ph = c_sf_phi[P][q * 8 + c + zo];
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
            dmma884(y0, y1, z[c][u][0], fPhiTB(0));
            dmma884(y0, y1, z[c][u][1], fPhiTB(1));
            *reinterpret_cast<double2*>(scr + u * kSfScrSlab + so_w) = make_double2(y0, y1);
          }
          __syncwarp();
          double y[2][2];
#pragma unroll
          for (int u = 0; u < 2; ++u) {
            const double b0 = scr[u * kSfScrSlab + so_r0], b1 = scr[u * kSfScrSlab + so_r1];
            y[u][0] = y[u][1] = 0.0;
            dmma884(y[u][0], y[u][1], fPhiTA(0), b0);
            dmma884(y[u][0], y[u][1], fPhiTA(1), b1);
          }
          // lane (g, t): nodes (a = g, b = 2t + e, c); the result overwrites the two columns:  s_l y_l - c x_l [first]
#pragma unroll
          for (int e = 0; e < 2; ++e) {
            const int bi = 2 * t + e;
            if (g < n1 && bi < n1) {
              const int l = g + n1 * bi + nn * c;
              S* xp = reinterpret_cast<S*>(xt + sf_pair_off<S>(l, pp));
              const double sl = sl_s[l];
              const double sh = idx_s[l] < 0 ? cshift : 0.0;          // the shift rides on the first contribution to the dof
              const double2 xo = sf_ld_pair(xp);
              sf_st_pair(xp, fma(sl, y[0][e], -sh * xo.x), fma(sl, y[1][e], -sh * xo.y));
            }
          }
        }
        __syncwarp();
      }
      // this warp's columns of the tile are final: hand them to the assembler warps (and, later, to the TMA)
      asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
      __syncwarp();
      if (lane == 0) mbar_arrive(bar_done + b);
      set = (set == 2) ? 0 : set + 1;
    }
#undef fPhiA
#undef fPhiB
#undef fDA
#undef fDB
#undef fDtA
#undef fDtB
#undef fPhiTA
#undef fPhiTB
  } else {
    asm volatile("setmaxnreg.dec.sync.aligned.u32 %0;" ::"n"(ws_regs_helper<S>()));
    if (warp == kWsComputeWarps) {
      // ===========================================================================================================
      // producer warp
      // ===========================================================================================================
      // index list + M^-1/2 of the cell of ticket tk into small set s (lane 0)
      auto issue_small = [&](long long tk, int s) {
        const int cell_l = pd.pos_cell[(int)(tk / nct)];
        unsigned char* dst = smem_dyn + L::off_small + s * L::small_bytes;
        const uint32_t nb = KP ? (uint32_t)mpad * 4u : (uint32_t)a.ktot[cell_l] * 4u;   // mpad + round8(projectors of the cell) entries
        mbar_expect_tx(bar_small + s, nb + (uint32_t)mpad * 8u);
        bulk_g2s(dst, a.gidx + a.idx_off[cell_l], nb, bar_small + s);
        bulk_g2s(dst + L::idx_stride * 4, sf.sloc + (int64_t)cell_l * mpad, (uint32_t)mpad * 8u, bar_small + s);
      };
      long long tk = 0;
      if (lane == 0) {
        tk = (long long)(atomicAdd(pd.counter, 1ull) - pd.ticket_base);
        ticket_s[0] = tk;
        if (tk < n_tiles) issue_small(tk, 0);
      }
      tk = __shfl_sync(0xffffffffu, tk, 0);
      int set = 0;
      for (int iter = 0;; ++iter) {
        const int b = iter & 1;
        if (iter >= 2) mbar_wait(bar_free + b, (uint32_t)((iter >> 1) - 1) & 1u);   // tile iter - 2 assembled
        if (tk >= n_tiles) {                                 // the end ticket: the other warps wake up, see it and leave
          if (lane == 0) mbar_arrive(bar_full + b);
          break;
        }
        const int cell_l = pd.pos_cell[(int)(tk / nct)];
        const int col0_l = (int)(tk % nct) * TN;
        const int64_t cp0 = sf.cell_proj_ptr[cell_l];
        const int np = KP ? 0 : (int)(sf.cell_proj_ptr[cell_l + 1] - cp0);
        const int npc = min(np, kSfCrowChunk), np8 = (np + 7) / 8 * 8;
        mbar_wait(bar_small + set, (uint32_t)(iter / 3) & 1u);
        const int32_t* idx_l = reinterpret_cast<const int32_t*>(smem_dyn + L::off_small + set * L::small_bytes);
        unsigned char* xt = smem_dyn + L::off_xt + b * L::tile_bytes;
        if (lane == 0) {
          asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
          mbar_expect_tx(bar_full + b, (uint32_t)mpad * 128u + (uint32_t)L::coef_bytes + (uint32_t)(npc * mpad * 8) +
                                           (uint32_t)np8 * 128u);
          bulk_g2s(smem_dyn + L::off_coef + b * L::coef_bytes, sf.coef + (int64_t)cell_l * L::coef_elems, (uint32_t)L::coef_bytes,
                   bar_full + b);
          if (np > 0)
            bulk_g2s(smem_dyn + L::off_crow + b * L::crow_bytes, sf.crows + cp0 * mpad, (uint32_t)(npc * mpad * 8), bar_full + b);
        }
        __syncwarp();
        for (int r4 = lane; r4 < mpad / 4; r4 += 32)
          tma_gather4(xt + (size_t)r4 * 512, &tmX, col0_l, idx_l[4 * r4] & 0x7fffffff, idx_l[4 * r4 + 1] & 0x7fffffff,
                      idx_l[4 * r4 + 2] & 0x7fffffff, idx_l[4 * r4 + 3] & 0x7fffffff, bar_full + b);
        if (lane < np8 / 4)                                  // rows of P of the cell's projectors (unused slots: the zero row)
          tma_gather4(smem_dyn + L::off_ps + b * L::ps_bytes + lane * 512, &tmP, col0_l, idx_l[mpad + 4 * lane],
                      idx_l[mpad + 4 * lane + 1], idx_l[mpad + 4 * lane + 2], idx_l[mpad + 4 * lane + 3], bar_full + b);
        // next ticket, and its small data one tile ahead (set (iter + 1) % 3 was last used by tile iter - 2: assembled)
        set = (set == 2) ? 0 : set + 1;
        if (lane == 0) {
          tk = (long long)(atomicAdd(pd.counter, 1ull) - pd.ticket_base);
          ticket_s[(iter + 1) & 3] = tk;
          if (tk < n_tiles) issue_small(tk, set);
        }
        tk = __shfl_sync(0xffffffffu, tk, 0);
      }
    } else {
      // ===========================================================================================================
      // assembler warps
      // ===========================================================================================================
      const int aw = warp - kWsComputeWarps - 1;
      const bool all_add = a.atomic || a.accumulate;
      const double alpha = (double)a.alpha;
      int set = 0;
      uint32_t phase_c2 = 0;
      for (int iter = 0;; ++iter) {
        const int b = iter & 1;
        mbar_wait(bar_full + b, (uint32_t)(iter >> 1) & 1u);
        const long long ticket = ticket_s[iter & 3];
        if (ticket >= n_tiles) break;
        mbar_wait(bar_small + set, (uint32_t)(iter / 3) & 1u);
        const int pos = (int)(ticket / nct), jt = (int)(ticket % nct);
        const int cell = pd.pos_cell[pos];
        const int col0 = jt * TN;
        const int ncols = min(TN, a.B - col0);
        const int64_t cp0 = sf.cell_proj_ptr[cell];
        const int np = KP ? 0 : (int)(sf.cell_proj_ptr[cell + 1] - cp0);
        const int npc = min(np, kSfCrowChunk);
        const unsigned char* xt = smem_dyn + L::off_xt + b * L::tile_bytes;
        const double* crow_s = reinterpret_cast<const double*>(smem_dyn + L::off_crow + b * L::crow_bytes);
        const S* Ps = reinterpret_cast<const S*>(smem_dyn + L::off_ps + b * L::ps_bytes);
        const int32_t* idx_s = reinterpret_cast<const int32_t*>(smem_dyn + L::off_small + set * L::small_bytes);
        if (!a.atomic && aw == 0) {                          // contributions of earlier cells to this tile's dofs are in memory
          const int d0 = pd.dep_ptr[pos], nd = pd.dep_ptr[pos + 1] - d0;
          for (int d = lane; d < nd; d += 32) {
            const uint32_t* f = pd.flags + (int64_t)pd.dep_pos[d0 + d] * nct + jt;
            while (ld_acquire_gpu(f) != pd.epoch) __nanosleep(64);
          }
        }
        mbar_wait(bar_done + b, (uint32_t)(iter >> 1) & 1u);  // the tile holds H~^loc X - c X [first]; its fields are dead
        // cells touched by two atoms: projector columns 8 .. np-1 arrive in place of the fields
        const int np2 = np > kSfCrowChunk ? np - kSfCrowChunk : 0;
        const double* crow2_s = reinterpret_cast<const double*>(smem_dyn + L::off_coef + b * L::coef_bytes);
        if (np2 > 0 && aw == 0 && lane == 0) {
          asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
          mbar_expect_tx(bar_crow2, (uint32_t)(np2 * mpad * 8));
          bulk_g2s(const_cast<double*>(crow2_s), sf.crows + (cp0 + kSfCrowChunk) * mpad, (uint32_t)(np2 * mpad * 8), bar_crow2);
        }
        ws_asm_sync();
        if (np2 > 0) { mbar_wait(bar_crow2, phase_c2); phase_c2 ^= 1u; }
        {
          // thread mapping = C fragment of an m8n8 tile: warp step = 8 rows (r = 8 mt + g) x TN columns, lane holds columns
          // 8 nt + 2t + {0, 1} of every 8-column block nt; two such steps are in flight per warp (the chain LDS -> DMMA ->
          // DMMA -> scale -> red of one step is pure latency).
          constexpr int nmt = (mc + 7) / 8;
          constexpr int kU = NT == 2 ? 2 : 1;               // FP32 tiles (32 columns) have four blocks per step already
#pragma unroll 1
          for (int mt0 = aw; mt0 < nmt; mt0 += kU * kWsAsmWarps) {
            double v[kU][NT][2], ca[kU][4];
            int idx[kU];
#pragma unroll
            for (int h = 0; h < kU; ++h) {
              const int mt = min(mt0 + h * kWsAsmWarps, nmt - 1);
              const int r = 8 * mt + g;                      // < mpad: the padding rows of the tile exist (never stored)
#pragma unroll
              for (int nt = 0; nt < NT; ++nt) {
                const double2 x2 = sf_ld_pair(reinterpret_cast<const S*>(xt + sf_pair_off<S>(r, 4 * nt + t)));
                v[h][nt][0] = x2.x; v[h][nt][1] = x2.y;
              }
              ca[h][0] = ca[h][1] = ca[h][2] = ca[h][3] = 0.0;
              if (np > 0) {
                if (t < npc) ca[h][0] = crow_s[t * mpad + r];
                if (4 + t < npc) ca[h][1] = crow_s[(4 + t) * mpad + r];
                if (t < np2) ca[h][2] = crow2_s[t * mpad + r];
                if (4 + t < np2) ca[h][3] = crow2_s[(4 + t) * mpad + r];
              }
              idx[h] = (r < mc) ? idx_s[r] : 0;
            }
            if (np > 0) {
#pragma unroll
              for (int nt = 0; nt < NT; ++nt) {
                const double p0 = (double)Ps[t * TN + 8 * nt + g], p1 = (double)Ps[(4 + t) * TN + 8 * nt + g];
#pragma unroll
                for (int h = 0; h < kU; ++h) {
                  dmma884(v[h][nt][0], v[h][nt][1], ca[h][0], p0);     // += sum_j C~[r][j] P[j][col]
                  dmma884(v[h][nt][0], v[h][nt][1], ca[h][1], p1);
                }
              }
              if (np2 > 0) {
#pragma unroll
                for (int nt = 0; nt < NT; ++nt) {
                  const double p2 = (double)Ps[(8 + t) * TN + 8 * nt + g], p3 = (double)Ps[(12 + t) * TN + 8 * nt + g];
#pragma unroll
                  for (int h = 0; h < kU; ++h) {
                    dmma884(v[h][nt][0], v[h][nt][1], ca[h][2], p2);
                    dmma884(v[h][nt][0], v[h][nt][1], ca[h][3], p3);
                  }
                }
              }
            }
#pragma unroll
            for (int h = 0; h < kU; ++h) {
              const int mt = mt0 + h * kWsAsmWarps;
              const int r = 8 * mt + g;
              if (mt >= nmt || r >= mc) continue;
              S* trow = a.Tg + (int64_t)(idx[h] & 0x7fffffff) * a.ldt + col0 + 2 * t;
              const bool add = all_add || idx[h] >= 0;
#pragma unroll
              for (int nt = 0; nt < NT; ++nt) {
                if (8 * nt + 2 * t >= ncols) continue;
                if (add) {
                  atomicAdd(trow + 8 * nt, (S)(alpha * v[h][nt][0]));
                  atomicAdd(trow + 8 * nt + 1, (S)(alpha * v[h][nt][1]));
                } else {
                  sf_st_pair(trow + 8 * nt, alpha * v[h][nt][0], alpha * v[h][nt][1]);
                }
              }
            }
          }
        }
        asm volatile("fence.proxy.async.shared::cta;" ::: "memory");   // generic reads of the buffers before the next TMA writes
        // tile assembled.  The release below is cumulative: the stores / reds of all assembler threads happen before this
        // barrier, hence before the st.release.gpu of the one thread that publishes the flag.
        ws_asm_sync();
        if (aw == 0 && lane == 0) {
          if (!a.atomic) st_release_gpu(pd.flags + (int64_t)pos * nct + jt, pd.epoch);
          mbar_arrive(bar_free + b);
        }
        set = (set == 2) ? 0 : set + 1;
      }
    }
  }
}
