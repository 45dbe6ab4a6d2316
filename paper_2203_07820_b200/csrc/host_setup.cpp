// Host-side setup of libchfsi: 1-D quadrature / basis tables, mesh validation, diagonal GLL mass matrix,
// graph colouring of the cells for the deterministic assembly, and the per-cell index / matrix layout.
//
// PAPER.md:301 (spectral FE on GLL nodes), PAPER.md:336 (GLL quadrature => diagonal M),
// PAPER.md:513-517 (cell-level extraction / assembly; C^{c_i} of size M_cell x N_psp^{c_i}),
// Alg. 4 step 3 (assembly of the projector coefficients over the cells of a projector).
#include <algorithm>
#include <cmath>
#include <cstring>
#include <map>

#include "common.h"

namespace chfsi {

namespace {

// P_n(x) and P_n'(x) in long double (Bonnet recurrence; derivative from (x^2-1) P_n' = n (x P_n - P_{n-1})).
void legendre_ld(int n, long double x, long double* pn, long double* dpn) {
  long double p0 = 1.0L, p1 = x;
  if (n == 0) { *pn = 1.0L; *dpn = 0.0L; return; }
  for (int k = 2; k <= n; ++k) {
    long double p2 = ((2 * k - 1) * x * p1 - (k - 1) * p0) / k;
    p0 = p1; p1 = p2;
  }
  *pn = p1;
  *dpn = n * (x * p1 - p0) / (x * x - 1.0L);
}

const long double kPi = 3.141592653589793238462643383279502884L;

void gauss_rule(int n, std::vector<double>* xs, std::vector<double>* ws) {
  xs->assign(n, 0.0); ws->assign(n, 0.0);
  for (int i = 0; i < n; ++i) {
    long double x = -cosl(kPi * (i + 0.75L) / (n + 0.5L));
    for (int it = 0; it < 100; ++it) {
      long double pn, dpn; legendre_ld(n, x, &pn, &dpn);
      long double dx = pn / dpn; x -= dx;
      if (fabsl(dx) < 1e-19L) break;
    }
    long double pn, dpn; legendre_ld(n, x, &pn, &dpn);
    (*xs)[i] = (double)x;
    (*ws)[i] = (double)(2.0L / ((1.0L - x * x) * dpn * dpn));
  }
}

void lobatto_rule(int p, std::vector<double>* xs, std::vector<double>* ws) {
  int n = p + 1;
  xs->assign(n, 0.0); ws->assign(n, 0.0);
  for (int i = 0; i < n; ++i) {
    long double x;
    if (i == 0) x = -1.0L;
    else if (i == p) x = 1.0L;
    else {
      x = -cosl(kPi * i / p);
      for (int it = 0; it < 100; ++it) {
        // f = P_p'(x); f' = P_p''(x) = (2x P_p' - p(p+1) P_p)/(1-x^2)   (Legendre's equation)
        long double pn, dpn; legendre_ld(p, x, &pn, &dpn);
        long double d2 = (2 * x * dpn - (long double)p * (p + 1) * pn) / (1.0L - x * x);
        long double dx = dpn / d2; x -= dx;
        if (fabsl(dx) < 1e-19L) break;
      }
    }
    long double pn, dpn;
    if (i == 0 || i == p) { pn = (i == 0 && (p & 1)) ? -1.0L : 1.0L; }
    else legendre_ld(p, x, &pn, &dpn);
    (*xs)[i] = (double)x;
    (*ws)[i] = (double)(2.0L / ((long double)p * (p + 1) * pn * pn));
  }
  // enforce exact antisymmetry of the nodes
  for (int i = 0; i < n / 2; ++i) { double v = 0.5 * ((*xs)[n - 1 - i] - (*xs)[i]); (*xs)[i] = -v; (*xs)[n - 1 - i] = v; }
  if (n & 1) (*xs)[n / 2] = 0.0;
}

}  // namespace

void build_tables(int p, Tables1D* t) {
  t->p = p; t->n1 = p + 1; t->nq1 = p + 2;
  lobatto_rule(p, &t->gll_x, &t->gll_w);
  gauss_rule(p + 2, &t->gq_x, &t->gq_w);
  int n1 = t->n1, nq1 = t->nq1;
  t->phi.assign((size_t)nq1 * n1, 0.0);
  t->dphi.assign((size_t)nq1 * n1, 0.0);
  // barycentric weights
  std::vector<long double> lam(n1, 1.0L);
  for (int i = 0; i < n1; ++i)
    for (int j = 0; j < n1; ++j)
      if (j != i) lam[i] /= ((long double)t->gll_x[i] - (long double)t->gll_x[j]);
  for (int q = 0; q < nq1; ++q) {
    long double x = t->gq_x[q];
    for (int i = 0; i < n1; ++i) {
      // l_i(x) = lam_i prod_{j != i} (x - x_j);  l_i'(x) = lam_i sum_{k != i} prod_{j != i,k} (x - x_j)
      long double val = lam[i], der = 0.0L;
      for (int j = 0; j < n1; ++j) if (j != i) val *= (x - (long double)t->gll_x[j]);
      for (int k = 0; k < n1; ++k) {
        if (k == i) continue;
        long double term = lam[i];
        for (int j = 0; j < n1; ++j) if (j != i && j != k) term *= (x - (long double)t->gll_x[j]);
        der += term;
      }
      t->phi[(size_t)q * n1 + i] = (double)val;
      t->dphi[(size_t)q * n1 + i] = (double)der;
    }
  }
}

namespace {
// det of the trilinear map's Jacobian at reference point (x,y,z); verts [8][3], v = vx + 2 vy + 4 vz.
double trilinear_detJ(const double* verts, double x, double y, double z) {
  double J[3][3] = {{0, 0, 0}, {0, 0, 0}, {0, 0, 0}};
  for (int v = 0; v < 8; ++v) {
    double sx = (v & 1) ? 1.0 : -1.0, sy = (v & 2) ? 1.0 : -1.0, sz = (v & 4) ? 1.0 : -1.0;
    double fx = 0.5 * (1.0 + sx * x), fy = 0.5 * (1.0 + sy * y), fz = 0.5 * (1.0 + sz * z);
    double g[3] = {0.5 * sx * fy * fz, fx * 0.5 * sy * fz, fx * fy * 0.5 * sz};
    for (int i = 0; i < 3; ++i)
      for (int d = 0; d < 3; ++d) J[i][d] += verts[v * 3 + i] * g[d];
  }
  return J[0][0] * (J[1][1] * J[2][2] - J[1][2] * J[2][1]) - J[0][1] * (J[1][0] * J[2][2] - J[1][2] * J[2][0]) +
         J[0][2] * (J[1][0] * J[2][1] - J[1][1] * J[2][0]);
}
}  // namespace

// M_g = sum over the cells of dof g of w_a w_b w_c detJ at the node: GLL quadrature makes the mass diagonal.
// Dofs and Jacobians are assumed valid as far as analyse_mesh checks them first; a non-positive Jacobian is reported.
std::string mesh_mass(const chfsi_mesh& mesh, const Tables1D& tab, std::vector<double>* mass) {
  const int n1 = tab.n1, mc = n1 * n1 * n1;
  mass->assign((size_t)mesh.n_dofs, 0.0);
  for (int64_t c = 0; c < mesh.n_cells; ++c) {
    const int32_t* cd = mesh.cell_dofs + c * mc;
    const double* vt = mesh.cell_vertices + c * 24;
    for (int k = 0; k < n1; ++k)
      for (int j = 0; j < n1; ++j)
        for (int i = 0; i < n1; ++i) {
          const int32_t g = cd[i + n1 * (j + n1 * k)];
          if (g < 0 || g >= mesh.n_dofs) return "cell " + std::to_string(c) + ": dof index out of range";
          double dj = trilinear_detJ(vt, tab.gll_x[i], tab.gll_x[j], tab.gll_x[k]);
          if (!(dj > 0.0)) return "cell " + std::to_string(c) + ": non-positive Jacobian";
          (*mass)[g] += tab.gll_w[i] * tab.gll_w[j] * tab.gll_w[k] * dj;
        }
  }
  return "";
}

std::string analyse_mesh(const chfsi_mesh& mesh, const chfsi_nonlocal* nl, const Tables1D& tab, int lda, int n_parts,
                         HostPlan* plan) {
  const int n1 = tab.n1, mc = n1 * n1 * n1;
  const int64_t nc = mesh.n_cells, nd = mesh.n_dofs;
  const int64_t n_proj = (nl && nl->n_proj > 0) ? nl->n_proj : 0;

  // ---- validation of the connectivity + dof -> cells incidence -------------------------------------------
  std::vector<int64_t> stamp(nd, -1);
  std::vector<int32_t> deg(nd, 0);
  for (int64_t c = 0; c < nc; ++c) {
    const int32_t* cd = mesh.cell_dofs + c * mc;
    for (int l = 0; l < mc; ++l) {
      int32_t g = cd[l];
      if (g < 0 || g >= nd) return "cell " + std::to_string(c) + ": dof index out of range";
      if (stamp[g] == c) return "cell " + std::to_string(c) + ": repeated dof inside one cell";
      stamp[g] = c; deg[g]++;
    }
  }
  for (int64_t g = 0; g < nd; ++g)
    if (deg[g] == 0) return "dof " + std::to_string(g) + " belongs to no cell";

  // ---- diagonal GLL mass, deterministic cell order ------------------------------------------
  {
    const std::string mm = mesh_mass(mesh, tab, &plan->mass);
    if (!mm.empty()) return mm;
  }

  // ---- greedy colouring of the cell graph (cells adjacent when they share a dof) ---------------------------
  std::vector<int64_t> dptr(nd + 1, 0);
  for (int64_t g = 0; g < nd; ++g) dptr[g + 1] = dptr[g] + deg[g];
  std::vector<int32_t> dcell(dptr[nd]);
  {
    std::vector<int64_t> cur(dptr.begin(), dptr.end() - 1);
    for (int64_t c = 0; c < nc; ++c)
      for (int l = 0; l < mc; ++l) dcell[cur[mesh.cell_dofs[c * mc + l]]++] = (int32_t)c;
  }
  std::vector<int32_t> color(nc, -1);
  std::vector<int64_t> used;  // used[col] == c  <=> colour taken by a neighbour of c
  int ncol = 0;
  for (int64_t c = 0; c < nc; ++c) {
    for (int l = 0; l < mc; ++l) {
      int32_t g = mesh.cell_dofs[c * mc + l];
      if (deg[g] == 1) continue;
      for (int64_t t = dptr[g]; t < dptr[g + 1]; ++t) {
        int32_t cc = color[dcell[t]];
        if (cc >= 0) { if ((size_t)cc >= used.size()) used.resize(cc + 1, -1); used[cc] = c; }
      }
    }
    int col = 0;
    while ((size_t)col < used.size() && used[col] == c) ++col;
    color[c] = col;
    if ((size_t)col >= used.size()) used.resize(col + 1, -1);
    ncol = std::max(ncol, col + 1);
  }
  plan->n_colors = ncol;
  plan->color_ptr.assign(ncol + 1, 0);
  for (int64_t c = 0; c < nc; ++c) plan->color_ptr[color[c] + 1]++;
  for (int k = 0; k < ncol; ++k) plan->color_ptr[k + 1] += plan->color_ptr[k];
  plan->color_cells.resize(nc);
  {
    std::vector<int32_t> cur(plan->color_ptr.begin(), plan->color_ptr.end() - 1);
    for (int64_t c = 0; c < nc; ++c) plan->color_cells[cur[color[c]]++] = (int32_t)c;
  }

  // ---- assembly dependencies: for the cell at position t of the colour order, the earlier positions whose
  // cells share a dof with it (they differ in colour).  The single-launch kernel orders the read-modify-writes
  // of a dof by waiting for these cells' completion flags, which fixes the summation order (= colour order).
  {
    std::vector<int32_t> pos(nc);
    for (int64_t t = 0; t < nc; ++t) pos[plan->color_cells[t]] = (int32_t)t;
    std::vector<int64_t> mark(nc, -1);
    plan->dep_ptr.assign(nc + 1, 0);
    plan->dep_pos.clear();
    for (int64_t t = 0; t < nc; ++t) {
      const int64_t c = plan->color_cells[t];
      for (int l = 0; l < mc; ++l) {
        int32_t g = mesh.cell_dofs[c * mc + l];
        if (deg[g] == 1) continue;
        for (int64_t u = dptr[g]; u < dptr[g + 1]; ++u) {
          int32_t cc = dcell[u];
          if (cc == c || mark[cc] == t) continue;
          mark[cc] = t;
          if (pos[cc] < t) plan->dep_pos.push_back(pos[cc]);
        }
      }
      std::sort(plan->dep_pos.begin() + plan->dep_ptr[t], plan->dep_pos.end());
      plan->dep_ptr[t + 1] = (int32_t)plan->dep_pos.size();
    }
  }

  // ---- cell-centric projector lists -------------------------------------------------------------------------
  plan->cell_proj_ptr.assign(nc + 1, 0);
  int64_t nnz = 0;
  if (n_proj) {
    nnz = nl->proj_cell_ptr[n_proj];
    if (nl->proj_cell_ptr[0] != 0 || nnz < 0) return "projector CSR: bad row pointers";
    for (int64_t j = 0; j < n_proj; ++j) {
      if (nl->proj_cell_ptr[j + 1] < nl->proj_cell_ptr[j]) return "projector CSR: row pointers not monotone";
      for (int64_t k = nl->proj_cell_ptr[j]; k < nl->proj_cell_ptr[j + 1]; ++k) {
        int32_t c = nl->proj_cell_idx[k];
        if (c < 0 || c >= nc) return "projector " + std::to_string(j) + ": cell index out of range";
        plan->cell_proj_ptr[c + 1]++;
      }
    }
  }
  for (int64_t c = 0; c < nc; ++c) plan->cell_proj_ptr[c + 1] += plan->cell_proj_ptr[c];
  plan->cell_proj_idx.assign(nnz, 0);
  plan->cell_proj_src.assign(nnz, 0);
  plan->proj_ptr.assign(n_proj + 1, 0);
  plan->proj_pcrow.assign(nnz, 0);
  if (n_proj) {
    std::vector<int64_t> cur(plan->cell_proj_ptr.begin(), plan->cell_proj_ptr.end() - 1);
    std::vector<int64_t> last(nc, -1);
    for (int64_t j = 0; j < n_proj; ++j) {
      plan->proj_ptr[j] = nl->proj_cell_ptr[j];
      for (int64_t k = nl->proj_cell_ptr[j]; k < nl->proj_cell_ptr[j + 1]; ++k) {
        int32_t c = nl->proj_cell_idx[k];
        if (last[c] == j) return "projector " + std::to_string(j) + ": cell listed twice";
        last[c] = j;
        int64_t row = cur[c]++;
        plan->cell_proj_idx[row] = (int32_t)j;
        plan->cell_proj_src[row] = k;
        plan->proj_pcrow[k] = row;
      }
    }
    plan->proj_ptr[n_proj] = nnz;
  }
  plan->pc_cells.clear();
  for (int64_t c = 0; c < nc; ++c)
    if (plan->cell_proj_ptr[c + 1] > plan->cell_proj_ptr[c]) plan->pc_cells.push_back((int32_t)c);

  // ---- dof-centric projector groups (same support = same atom), their dof rows and the CTA segments --------
  plan->n_groups = 0;
  plan->grp_row_ptr.assign(1, 0);
  plan->grow_dof.clear(); plan->grp_proj.clear();
  plan->seg_ptr.assign(1, 0); plan->grp_seg_ptr.assign(1, 0);
  plan->proj_grp.assign(n_proj, 0); plan->proj_slot.assign(n_proj, 0);
  if (n_proj) {
    std::map<std::vector<int32_t>, std::vector<int32_t>> by_support;   // ordered: deterministic group numbering
    for (int64_t j = 0; j < n_proj; ++j) {
      std::vector<int32_t> cells(nl->proj_cell_idx + nl->proj_cell_ptr[j], nl->proj_cell_idx + nl->proj_cell_ptr[j + 1]);
      std::sort(cells.begin(), cells.end());
      by_support[cells].push_back((int32_t)j);
    }
    std::vector<uint8_t> in_grp(nd, 0);
    for (const auto& kv : by_support) {
      const std::vector<int32_t>& cells = kv.first;
      if (cells.empty()) {   // projector without support: its coefficient is zero; give it an empty group
        for (int32_t j : kv.second) { plan->proj_grp[j] = -1; plan->proj_slot[j] = 0; }
        continue;
      }
      std::vector<int32_t> dofs;
      for (int32_t c : cells)
        for (int l = 0; l < mc; ++l) {
          int32_t g = mesh.cell_dofs[(int64_t)c * mc + l];
          if (!in_grp[g]) { in_grp[g] = 1; dofs.push_back(g); }
        }
      std::sort(dofs.begin(), dofs.end());
      for (int32_t g : dofs) in_grp[g] = 0;
      for (size_t i0 = 0; i0 < kv.second.size(); i0 += kProjGroup) {
        const int grp = plan->n_groups++;
        const size_t ni = std::min<size_t>(kProjGroup, kv.second.size() - i0);
        for (int i = 0; i < kProjGroup; ++i) plan->grp_proj.push_back((size_t)i < ni ? kv.second[i0 + i] : -1);
        for (size_t i = 0; i < ni; ++i) { plan->proj_grp[kv.second[i0 + i]] = grp; plan->proj_slot[kv.second[i0 + i]] = (int32_t)i; }
        const int32_t r0 = (int32_t)plan->grow_dof.size();
        plan->grow_dof.insert(plan->grow_dof.end(), dofs.begin(), dofs.end());
        const int32_t r1 = (int32_t)plan->grow_dof.size();
        plan->grp_row_ptr.push_back(r1);
        for (int32_t r = r0; r < r1; r += kProjSegRows) plan->seg_ptr.push_back(std::min(r1, r + kProjSegRows));
        plan->grp_seg_ptr.push_back((int32_t)plan->seg_ptr.size() - 1);
      }
    }
  }

  // ---- per-cell layout: K_c, matrix offsets, gather/scatter index lists with first-contribution flags --------
  // rows 0..mc-1: nodes; rows mc..mpad-1: padding (zero matrix rows, gather any valid dof); rows mpad..: projectors.
  // Node rows and projector rows never share a group of 4 (or a panel of 8) rows, so every TMA row gather of the
  // contraction kernel reads from ONE array (X or P).
  const int mpad = (mc + 7) / 8 * 8;
  plan->ktot.resize(nc);
  plan->mat_off.assign(nc + 1, 0);
  plan->idx_off.assign(nc + 1, 0);
  for (int64_t c = 0; c < nc; ++c) {
    int64_t np = plan->cell_proj_ptr[c + 1] - plan->cell_proj_ptr[c];
    int kt = (int)(mpad + (np + 7) / 8 * 8);
    plan->ktot[c] = kt;
    plan->mat_off[c + 1] = plan->mat_off[c] + (int64_t)n_parts * kt * lda;
    plan->idx_off[c + 1] = plan->idx_off[c] + kt;
  }
  plan->gidx.assign(plan->idx_off[nc], (int32_t)n_proj);
  for (int64_t c = 0; c < nc; ++c) {
    int32_t* gi = plan->gidx.data() + plan->idx_off[c];
    for (int l = 0; l < mc; ++l) gi[l] = mesh.cell_dofs[c * mc + l];
    for (int l = mc; l < mpad; ++l) gi[l] = mesh.cell_dofs[c * mc];
    int64_t np = plan->cell_proj_ptr[c + 1] - plan->cell_proj_ptr[c];
    for (int64_t i = 0; i < np; ++i) gi[mpad + i] = plan->cell_proj_idx[plan->cell_proj_ptr[c] + i];
  }
  std::vector<uint8_t> seen(nd, 0);
  for (int64_t t = 0; t < nc; ++t) {
    int64_t c = plan->color_cells[t];
    int32_t* gi = plan->gidx.data() + plan->idx_off[c];
    for (int l = 0; l < mc; ++l) {
      int32_t g = gi[l];
      if (!seen[g]) { seen[g] = 1; gi[l] = (int32_t)((uint32_t)g | kFirstBit); }
    }
  }
  return "";
}

}  // namespace chfsi
