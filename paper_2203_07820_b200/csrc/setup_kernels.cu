// Setup kernels of libchfsi (untimed, once per operator): the Loewdin-scaled cell matrices
//
//   mat[c][k][m] = s_k ( 1/2 K^e_km + V^e_km ) s_m                          k, m < M_cell
//   K^e_km = sum_q w_q detJ_q (J_q^-T grad N_k)(q) . (J_q^-T grad N_m)(q)   Eq. 30 term 1
//   V^e_km = sum_q w_q detJ_q V_eff(q) N_k(q) N_m(q)                         Eq. 40 (with
//                                                                            P_Ip = N_j N_k as PAPER.md:470 says)
//   mat[c][M_cell+i][m] = s_m sum_q w_q detJ_q chi_j(q) N_m(q)               Eq. 33, Gamma point
//
// with s = M^-1/2 (Eq. 34; the paper folds it into the cell matrices).
//
// The quadrature sums are evaluated by sum factorisation over the tensor-product structure
// N_k(q) = phi_a(qa) phi_b(qb) phi_c(qc):  every one of the 10 weight fields (V and the 9 entries of the
// metric tensor w detJ J^-1 J^-T) costs three 1-D contractions instead of a dense (M_cell^2 x n_q) product.
#include <cstdio>

#include "common.h"

namespace chfsi {

namespace {

constexpr int kMaxNq1 = 10;

struct Geom {
  double detJ;
  double G[3][3];  // sum_i Jinv[a][i] Jinv[b][i]
  double Ji[3][3]; // Jinv[d][i] = d xi_d / d x_i
};

__device__ inline Geom trilinear_geom(const double* vt /*[8][3]*/, double x, double y, double z) {
  double J[3][3] = {{0, 0, 0}, {0, 0, 0}, {0, 0, 0}};
#pragma unroll
  for (int v = 0; v < 8; ++v) {
    double sx = (v & 1) ? 1.0 : -1.0, sy = (v & 2) ? 1.0 : -1.0, sz = (v & 4) ? 1.0 : -1.0;
    double fx = 0.5 * (1.0 + sx * x), fy = 0.5 * (1.0 + sy * y), fz = 0.5 * (1.0 + sz * z);
    double g0 = 0.5 * sx * fy * fz, g1 = fx * 0.5 * sy * fz, g2 = fx * fy * 0.5 * sz;
#pragma unroll
    for (int i = 0; i < 3; ++i) {
      double xv = vt[v * 3 + i];
      J[i][0] += xv * g0; J[i][1] += xv * g1; J[i][2] += xv * g2;
    }
  }
  Geom r;
  double c00 = J[1][1] * J[2][2] - J[1][2] * J[2][1];
  double c01 = J[1][2] * J[2][0] - J[1][0] * J[2][2];
  double c02 = J[1][0] * J[2][1] - J[1][1] * J[2][0];
  r.detJ = J[0][0] * c00 + J[0][1] * c01 + J[0][2] * c02;
  double id = 1.0 / r.detJ;
  // Jinv[d][i] = d xi_d / d x_i = cofactor(J)[i][d] / det
  double Ji[3][3];
  Ji[0][0] = c00 * id; Ji[1][0] = c01 * id; Ji[2][0] = c02 * id;
  Ji[0][1] = (J[0][2] * J[2][1] - J[0][1] * J[2][2]) * id;
  Ji[1][1] = (J[0][0] * J[2][2] - J[0][2] * J[2][0]) * id;
  Ji[2][1] = (J[0][1] * J[2][0] - J[0][0] * J[2][1]) * id;
  Ji[0][2] = (J[0][1] * J[1][2] - J[0][2] * J[1][1]) * id;
  Ji[1][2] = (J[0][2] * J[1][0] - J[0][0] * J[1][2]) * id;
  Ji[2][2] = (J[0][0] * J[1][1] - J[0][1] * J[1][0]) * id;
#pragma unroll
  for (int a = 0; a < 3; ++a)
#pragma unroll
    for (int b = 0; b < 3; ++b) {
      r.G[a][b] = Ji[a][0] * Ji[b][0] + Ji[a][1] * Ji[b][1] + Ji[a][2] * Ji[b][2];
      r.Ji[a][b] = Ji[a][b];
    }
  return r;
}

struct SetupTables {
  const double* pp;     // [4][nq1][n1*n1]  pair products f_a(q) g_a'(q); idx = (f is derivative) + 2 (g is derivative)
  const double* phi;    // [nq1][n1]
  const double* gq_x;   // [nq1]
  const double* gq_w;   // [nq1]
};

// One CTA loops over cells; scratch64 is a per-CTA [m_cell][m_cell] FP64 accumulator in global memory.
template <typename T>
__global__ void __launch_bounds__(256) k_cell_matrix(int n1, int nq1, int64_t n_cells, SetupTables tb,
                                                     const double* __restrict__ verts, const double* __restrict__ veff,
                                                     const int32_t* __restrict__ gidx, const int64_t* __restrict__ idx_off,
                                                     const int64_t* __restrict__ mat_off, const int32_t* __restrict__ ktot,
                                                     const double* __restrict__ mass, int lda, int mw, int n_parts,
                                                     T* __restrict__ mat, double* __restrict__ scratch64,
                                                     int* __restrict__ bad_flag, int zero_tail) {
  extern __shared__ double smem[];
  const int nn = n1 * n1, nq2 = nq1 * nq1, nq = nq1 * nq2, mc = n1 * nn;
  double* Wf = smem;                    // [10][nq]
  double* T1 = Wf + 10 * nq;            // [nn][nq2]
  double* PP = T1 + nn * nq2;           // [4][nq1][nn]
  double* vt = PP + 4 * nq1 * nn;       // [24]
  for (int i = threadIdx.x; i < 4 * nq1 * nn; i += blockDim.x) PP[i] = tb.pp[i];
  double* H64 = scratch64 + (size_t)blockIdx.x * mc * mc;

  for (int64_t c = blockIdx.x; c < n_cells; c += gridDim.x) {
    __syncthreads();
    if (threadIdx.x < 24) vt[threadIdx.x] = verts[c * 24 + threadIdx.x];
    __syncthreads();
    for (int q = threadIdx.x; q < nq; q += blockDim.x) {
      int qa = q % nq1, qb = (q / nq1) % nq1, qc = q / nq2;
      Geom g = trilinear_geom(vt, tb.gq_x[qa], tb.gq_x[qb], tb.gq_x[qc]);
      if (!(g.detJ > 0.0)) atomicExch(bad_flag, 1);
      double wj = tb.gq_w[qa] * tb.gq_w[qb] * tb.gq_w[qc] * g.detJ;
      Wf[q] = wj * veff[c * nq + q];
#pragma unroll
      for (int a = 0; a < 3; ++a)
#pragma unroll
        for (int b = 0; b < 3; ++b) Wf[(1 + 3 * a + b) * nq + q] = 0.5 * wj * g.G[a][b];
    }
    __syncthreads();
    for (int term = 0; term < 10; ++term) {
      int al = -1, be = -1;
      if (term > 0) { al = (term - 1) / 3; be = (term - 1) % 3; }
      const double* PPx = PP + ((al == 0 ? 1 : 0) + (be == 0 ? 2 : 0)) * nq1 * nn;
      const double* PPy = PP + ((al == 1 ? 1 : 0) + (be == 1 ? 2 : 0)) * nq1 * nn;
      const double* PPz = PP + ((al == 2 ? 1 : 0) + (be == 2 ? 2 : 0)) * nq1 * nn;
      const double* W = Wf + term * nq;
      // stage 1: T1[aa][qb,qc] = sum_qa W[qa,qb,qc] PPx[qa][aa]
      for (int o = threadIdx.x; o < nn * nq2; o += blockDim.x) {
        int aa = o / nq2, r = o % nq2;
        double s = 0.0;
        for (int qa = 0; qa < nq1; ++qa) s += W[qa + nq1 * r] * PPx[qa * nn + aa];
        T1[o] = s;
      }
      __syncthreads();
      // stages 2+3: item (aa, bb); t2[qc] = sum_qb T1[aa][qb,qc] PPy[qb][bb]; out[cc] = sum_qc t2[qc] PPz[qc][cc]
      for (int it = threadIdx.x; it < nn * nn; it += blockDim.x) {
        int aa = it % nn, bb = it / nn;
        int a = aa / n1, a2 = aa % n1, b = bb / n1, b2 = bb % n1;
        double t2[kMaxNq1];
        for (int qc = 0; qc < nq1; ++qc) {
          double s = 0.0;
          for (int qb = 0; qb < nq1; ++qb) s += T1[aa * nq2 + qb + nq1 * qc] * PPy[qb * nn + bb];
          t2[qc] = s;
        }
        for (int cc = 0; cc < nn; ++cc) {
          int cz = cc / n1, cz2 = cc % n1;
          double s = 0.0;
          for (int qc = 0; qc < nq1; ++qc) s += t2[qc] * PPz[qc * nn + cc];
          size_t k = a + n1 * (b + n1 * cz), m = a2 + n1 * (b2 + n1 * cz2);
          if (term == 0) H64[k * mc + m] = s; else H64[k * mc + m] += s;
        }
      }
      __syncthreads();
    }
    // Loewdin scaling (Eq. 34), conversion to T, zero padding of the Hamiltonian rows
    const int32_t* gi = gidx + idx_off[c];
    T* M = mat + mat_off[c];
    const int kc = ktot[c];
    for (int part = 0; part < n_parts; ++part) {
      T* Mp = M + (int64_t)part * kc * lda;
      for (int o = threadIdx.x; o < mc * lda; o += blockDim.x) {
        int k = o / lda, ml = o % lda, m = part * mw + ml;
        double v = 0.0;
        if (ml < mw && m < mc) {
          double sk = 1.0 / sqrt(mass[gi[k] & 0x7fffffff]), sm = 1.0 / sqrt(mass[gi[m] & 0x7fffffff]);
          v = H64[(size_t)k * mc + m] * sk * sm;
        }
        Mp[o] = (T)v;
      }
      // padding rows beyond the projector rows (and the projector rows themselves, filled later) start at zero
      if (zero_tail)
        for (int o = mc * lda + threadIdx.x; o < kc * lda; o += blockDim.x) Mp[o] = (T)0;
    }
  }
}

// One CTA per (cell, projector) row r of the cell-centric list:  C_m = sum_q w_q detJ_q chi(q) N_m(q).
template <typename T>
__global__ void __launch_bounds__(256) k_cell_projector(int n1, int nq1, SetupTables tb, const double* __restrict__ verts,
                                                        const double* __restrict__ chi, const int64_t* __restrict__ row_src,
                                                        const int32_t* __restrict__ row_cell,
                                                        const int64_t* __restrict__ cell_proj_ptr,
                                                        const int32_t* __restrict__ gidx, const int64_t* __restrict__ idx_off,
                                                        const int64_t* __restrict__ mat_off, const double* __restrict__ mass,
                                                        const int32_t* __restrict__ ktot, int lda, int mw, int n_parts,
                                                        T* __restrict__ mat) {
  extern __shared__ double smem[];
  const int nn = n1 * n1, nq2 = nq1 * nq1, nq = nq1 * nq2, mc = n1 * nn;
  double* W = smem;              // [nq]
  double* A = W + nq;            // [n1][nq2]   after contracting qa
  double* Bt = A + n1 * nq2;     // [nn][nq1]   after contracting qb
  double* ph = Bt + nn * nq1;    // [nq1][n1]
  double* vt = ph + nq1 * n1;    // [24]
  const int64_t r = blockIdx.x;
  const int64_t c = row_cell[r];
  const int64_t src = row_src[r];
  if (threadIdx.x < 24) vt[threadIdx.x] = verts[c * 24 + threadIdx.x];
  for (int i = threadIdx.x; i < nq1 * n1; i += blockDim.x) ph[i] = tb.phi[i];
  __syncthreads();
  for (int q = threadIdx.x; q < nq; q += blockDim.x) {
    int qa = q % nq1, qb = (q / nq1) % nq1, qc = q / nq2;
    Geom g = trilinear_geom(vt, tb.gq_x[qa], tb.gq_x[qb], tb.gq_x[qc]);
    W[q] = tb.gq_w[qa] * tb.gq_w[qb] * tb.gq_w[qc] * g.detJ * chi[src * nq + q];
  }
  __syncthreads();
  for (int o = threadIdx.x; o < n1 * nq2; o += blockDim.x) {   // A[a][qb,qc]
    int a = o / nq2, rr = o % nq2;
    double s = 0.0;
    for (int qa = 0; qa < nq1; ++qa) s += W[qa + nq1 * rr] * ph[qa * n1 + a];
    A[o] = s;
  }
  __syncthreads();
  for (int o = threadIdx.x; o < nn * nq1; o += blockDim.x) {   // Bt[a + n1 b][qc]
    int ab = o / nq1, qc = o % nq1, a = ab % n1, b = ab / n1;
    double s = 0.0;
    for (int qb = 0; qb < nq1; ++qb) s += A[a * nq2 + qb + nq1 * qc] * ph[qb * n1 + b];
    Bt[o] = s;
  }
  __syncthreads();
  const int32_t* gi = gidx + idx_off[c];
  const int krow = (mc + 7) / 8 * 8 + (int)(r - cell_proj_ptr[c]);
  const int kc = ktot[c];
  for (int o = threadIdx.x; o < n_parts * lda; o += blockDim.x) {
    const int part = o / lda, ml = o % lda, m = part * mw + ml;
    double v = 0.0;
    if (ml < mw && m < mc) {
      int ab = m % nn, cz = m / nn;
      for (int qc = 0; qc < nq1; ++qc) v += Bt[ab * nq1 + qc] * ph[qc * n1 + cz];
      v *= 1.0 / sqrt(mass[gi[m] & 0x7fffffff]);
    }
    mat[mat_off[c] + ((int64_t)part * kc + krow) * lda + ml] = (T)v;
  }
}

// Fields of the sum-factorised apply at the Gauss points of every cell, in the lane order of k_apply_sf:
//   coef[c][qc][k][lane = 4 qa + qb/2][e = qb % 2],  k = 0: w detJ V_eff;  k = 1..6: 1/2 w detJ (J^-1 J^-T)_{xx,xy,xz,yy,yz,zz}
// (the integrands of Eq. 40 / Eq. 30 term 1, before the shape functions are applied).  k-point variant
// (nf = 10): k = 7..9: w detJ (J^-1 kvec)_d, the integrand of the last term of Eq. 30 without its factor -i:
// k . grad_x u = sum_d (J^-1 kvec)_d d u / d xi_d.
__global__ void __launch_bounds__(256) k_sf_fields(int nq1, int nf, int64_t n_cells, SetupTables tb, const double* __restrict__ verts,
                                                   const double* __restrict__ veff, double kx, double ky, double kz,
                                                   double* __restrict__ coef) {
  __shared__ double vt[24];
  const int64_t c = blockIdx.x;
  const int nq2 = nq1 * nq1, nq = nq1 * nq2;
  if (threadIdx.x < 24) vt[threadIdx.x] = verts[c * 24 + threadIdx.x];
  __syncthreads();
  double* out = coef + c * (int64_t)nq1 * nf * 64;
  for (int q = threadIdx.x; q < nq; q += blockDim.x) {
    const int qa = q % nq1, qb = (q / nq1) % nq1, qc = q / nq2;
    const Geom g = trilinear_geom(vt, tb.gq_x[qa], tb.gq_x[qb], tb.gq_x[qc]);
    const double wj = tb.gq_w[qa] * tb.gq_w[qb] * tb.gq_w[qc] * g.detJ;
    const int slot = (4 * qa + (qb >> 1)) * 2 + (qb & 1);
    double* o = out + (int64_t)qc * nf * 64 + slot;
    o[0] = wj * veff[c * nq + q];
    o[64] = 0.5 * wj * g.G[0][0]; o[128] = 0.5 * wj * g.G[0][1]; o[192] = 0.5 * wj * g.G[0][2];
    o[256] = 0.5 * wj * g.G[1][1]; o[320] = 0.5 * wj * g.G[1][2]; o[384] = 0.5 * wj * g.G[2][2];
    if (nf == 10) {
      o[448] = wj * (g.Ji[0][0] * kx + g.Ji[0][1] * ky + g.Ji[0][2] * kz);
      o[512] = wj * (g.Ji[1][0] * kx + g.Ji[1][1] * ky + g.Ji[1][2] * kz);
      o[576] = wj * (g.Ji[2][0] * kx + g.Ji[2][1] * ky + g.Ji[2][2] * kz);
    }
  }
}

template <typename U>
cudaError_t upload(U** dst, const U* src, size_t n, cudaStream_t st) {
  *dst = nullptr;
  if (n == 0) n = 1;
  cudaError_t e = cudaMalloc((void**)dst, n * sizeof(U));
  if (e != cudaSuccess) return e;
  if (src) e = cudaMemcpyAsync(*dst, src, n * sizeof(U), cudaMemcpyHostToDevice, st);
  return e;
}

}  // namespace

#define CK(x) do { cudaError_t e_ = (x); if (e_ != cudaSuccess) { err = e_; goto done; } } while (0)

namespace {
// Hamiltonian rows of all cell matrices from V_eff at the Gauss points (host pointer); op->setup_* must exist.
cudaError_t launch_local_matrices(Op* op, const double* veff_host, cudaStream_t stream, int zero_tail, bool* bad_jacobian,
                                  const double* veff_dev = nullptr) {
  cudaError_t err = cudaSuccess;
  const int n1 = op->n1, nq1 = op->nq1, nn = n1 * n1, nq = nq1 * nq1 * nq1, mc = n1 * nn;
  const int64_t nc = op->n_cells;
  double *d_veff = nullptr, *d_scratch = nullptr, *d_veff_own = nullptr;
  int* d_bad = nullptr;
  int h_bad = 0;
  if (veff_dev) d_veff = const_cast<double*>(veff_dev);
  else { CK(upload(&d_veff_own, veff_host, (size_t)nc * nq, stream)); d_veff = d_veff_own; }
  CK(upload(&d_bad, &h_bad, 1, stream));
  {
    SetupTables tb{op->setup_pp, op->setup_phi, op->setup_gx, op->setup_gw};
    int grid = (int)std::min<int64_t>(nc, 296);
    CK(cudaMalloc((void**)&d_scratch, (size_t)grid * mc * mc * sizeof(double)));
    size_t smem = ((size_t)10 * nq + (size_t)nn * nq1 * nq1 + (size_t)4 * nq1 * nn + 24) * sizeof(double);
    if (op->precision == 64) {
      CK(cudaFuncSetAttribute(k_cell_matrix<double>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
      k_cell_matrix<double><<<grid, 256, smem, stream>>>(n1, nq1, nc, tb, op->setup_verts, d_veff, op->gidx, op->idx_off,
                                                         op->mat_off, op->ktot, op->mass, op->lda, op->mw, op->n_parts,
                                                         (double*)op->mat, d_scratch, d_bad, zero_tail);
    } else {
      CK(cudaFuncSetAttribute(k_cell_matrix<float>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
      k_cell_matrix<float><<<grid, 256, smem, stream>>>(n1, nq1, nc, tb, op->setup_verts, d_veff, op->gidx, op->idx_off,
                                                        op->mat_off, op->ktot, op->mass, op->lda, op->mw, op->n_parts,
                                                        (float*)op->mat, d_scratch, d_bad, zero_tail);
    }
    CK(cudaGetLastError());
    CK(cudaMemcpyAsync(&h_bad, d_bad, sizeof(int), cudaMemcpyDeviceToHost, stream));
    CK(cudaStreamSynchronize(stream));
    if (bad_jacobian) *bad_jacobian = (h_bad != 0);
  }
done:
  cudaFree(d_veff_own); cudaFree(d_scratch); cudaFree(d_bad);
  return err;
}
}  // namespace

cudaError_t build_sf_fields_dev(Op* op, const double* veff_q_dev, cudaStream_t stream) {
  cudaError_t err = cudaSuccess;
  const int nq1 = op->nq1;
  const int nf = op->kpoint ? 10 : 7;
  const size_t elems = (size_t)op->n_cells * nq1 * nf * 64;
  if (!op->sf_coef) {
    CK(cudaMalloc((void**)&op->sf_coef, elems * sizeof(double)));
    CK(cudaMemsetAsync(op->sf_coef, 0, elems * sizeof(double), stream));   // lanes beyond the Gauss grid (p < 6) stay zero
  }
  {
    SetupTables tb{op->setup_pp, op->setup_phi, op->setup_gx, op->setup_gw};
    k_sf_fields<<<(unsigned)op->n_cells, 256, 0, stream>>>(nq1, nf, op->n_cells, tb, op->setup_verts, veff_q_dev, op->kvec[0],
                                                           op->kvec[1], op->kvec[2], op->sf_coef);
    CK(cudaGetLastError());
  }
done:
  return err;
}

cudaError_t build_sf_fields(Op* op, const double* veff_q_host, cudaStream_t stream) {
  cudaError_t err = cudaSuccess;
  double* d_veff = nullptr;
  CK(upload(&d_veff, veff_q_host, (size_t)op->n_cells * op->n_q, stream));
  CK(build_sf_fields_dev(op, d_veff, stream));
  CK(cudaStreamSynchronize(stream));
done:
  cudaFree(d_veff);
  return err;
}

cudaError_t refresh_dense_matrices(Op* op, cudaStream_t stream) {
  if (!op->dense_stale) return cudaSuccess;
  cudaError_t e = launch_local_matrices(op, nullptr, stream, /*zero_tail=*/0, nullptr, op->veff_dev);
  if (e != cudaSuccess) return e;
  if ((e = capture_diagonal(op, stream))) return e;
  op->dense_stale = false;
  op->launches += 2;
  return cudaSuccess;
}

cudaError_t rebuild_local_matrices(Op* op, const double* veff_q_host, cudaStream_t stream) {
  return launch_local_matrices(op, veff_q_host, stream, /*zero_tail=*/0, nullptr);
}

// Projector rows of the cell matrices, C^c_{l,j} = sum_q w detJ chi_j(q) N_l(q) (Eq. 33), from the samples
// chi (HOST pointer [nnz][(p+2)^3]); op->setup_* must exist.  The k-point variant calls it a second time with the
// imaginary parts of the samples.  Synchronises the stream.
cudaError_t build_cell_projectors(Op* op, const HostPlan& plan, const double* chi_host, cudaStream_t stream) {
  cudaError_t err = cudaSuccess;
  const int n1 = op->n1, nq1 = op->nq1, nn = n1 * n1, nq = nq1 * nq1 * nq1;
  double* d_chi = nullptr;
  int64_t* d_row_src = nullptr; int32_t* d_row_cell = nullptr;
  std::vector<int32_t> row_cell(plan.cell_proj_idx.size());
  for (int64_t c = 0; c < op->n_cells; ++c)
    for (int64_t r = plan.cell_proj_ptr[c]; r < plan.cell_proj_ptr[c + 1]; ++r) row_cell[r] = (int32_t)c;
  {
    SetupTables tb{op->setup_pp, op->setup_phi, op->setup_gx, op->setup_gw};
    CK(upload(&d_chi, chi_host, (size_t)op->nnz_cp * nq, stream));
    CK(upload(&d_row_src, plan.cell_proj_src.data(), plan.cell_proj_src.size(), stream));
    CK(upload(&d_row_cell, row_cell.data(), row_cell.size(), stream));
    size_t smem2 = ((size_t)nq + (size_t)n1 * nq1 * nq1 + (size_t)nn * nq1 + (size_t)nq1 * n1 + 24) * sizeof(double);
    if (op->precision == 64)
      k_cell_projector<double><<<(unsigned)op->nnz_cp, 256, smem2, stream>>>(
          n1, nq1, tb, op->setup_verts, d_chi, d_row_src, d_row_cell, op->cell_proj_ptr, op->gidx, op->idx_off, op->mat_off,
          op->mass, op->ktot, op->lda, op->mw, op->n_parts, (double*)op->mat);
    else
      k_cell_projector<float><<<(unsigned)op->nnz_cp, 256, smem2, stream>>>(
          n1, nq1, tb, op->setup_verts, d_chi, d_row_src, d_row_cell, op->cell_proj_ptr, op->gidx, op->idx_off, op->mat_off,
          op->mass, op->ktot, op->lda, op->mw, op->n_parts, (float*)op->mat);
    CK(cudaGetLastError());
    CK(cudaStreamSynchronize(stream));
  }
done:
  cudaFree(d_chi); cudaFree(d_row_src); cudaFree(d_row_cell);
  return err;
}

cudaError_t build_cell_matrices(Op* op, const HostPlan& plan, const Tables1D& tab, const chfsi_mesh& mesh,
                                const chfsi_potential& pot, const chfsi_nonlocal* nl, cudaStream_t stream,
                                bool* bad_jacobian) {
  cudaError_t err = cudaSuccess;
  const int n1 = tab.n1, nq1 = tab.nq1, nn = n1 * n1, nq = nq1 * nq1 * nq1;
  const int64_t nc = op->n_cells;
  std::vector<double> pp((size_t)4 * nq1 * nn);
  for (int idx = 0; idx < 4; ++idx)
    for (int q = 0; q < nq1; ++q)
      for (int a = 0; a < n1; ++a)
        for (int a2 = 0; a2 < n1; ++a2) {
          double f = (idx & 1) ? tab.dphi[q * n1 + a] : tab.phi[q * n1 + a];
          double g = (idx & 2) ? tab.dphi[q * n1 + a2] : tab.phi[q * n1 + a2];
          pp[((size_t)idx * nq1 + q) * nn + a * n1 + a2] = f * g;
        }
  CK(upload(&op->setup_pp, pp.data(), pp.size(), stream));
  CK(upload(&op->setup_phi, tab.phi.data(), tab.phi.size(), stream));
  CK(upload(&op->setup_gx, tab.gq_x.data(), tab.gq_x.size(), stream));
  CK(upload(&op->setup_gw, tab.gq_w.data(), tab.gq_w.size(), stream));
  CK(upload(&op->setup_verts, mesh.cell_vertices, (size_t)nc * 24, stream));
  CK(launch_local_matrices(op, pot.veff_q, stream, /*zero_tail=*/1, bad_jacobian));
  if (op->nnz_cp > 0) CK(build_cell_projectors(op, plan, nl->chi_q, stream));
done:
  return err;
}

}  // namespace chfsi
