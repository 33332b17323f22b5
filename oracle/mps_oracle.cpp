// oracle/mps_oracle.cpp -- TEST INFRASTRUCTURE, NOT THE PRODUCT.
//
// Plain, slow, single-threaded C++17 CPU implementation of the MPS time-step
// particle-interaction path of arXiv 2105.01677 ("A Fluid Simulation System
// Based on the MPS Method"), written from the paper text only.  It is the
// oracle the CUDA path (paper_2105_01677_b200/csrc) is compared against and
// shares no code, header, table or helper with it.  Only tests/,
// __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs
// may load it.  Build: g++ -O2 -ffp-contract=off -shared -fPIC (oracle/build.py).
//
// Citations: "P:n" = /root/reference/PAPER.md line n.  "Qk" = reading k listed
// in DESIGN.md section 3 (where the paper is silent, ambiguous or garbled).
//
// Every function follows the paper's order and notation step by step; there is
// no blocking, fusion or reordering.  Particles stay in the caller's original
// order; the cell grid is used only to find neighbours (and to report the
// sort), and `brute` replaces it by the O(N^2) double loop that *defines* the
// fixed-radius neighbour set.
//
// Pins (tests/test_oracle_pins.py, -m "not gpu"): brute-force neighbour sets,
// hand-computed n0 / lambda shells, lattice densities, free-surface counts,
// Laplacian of a quadratic, gradient of a linear field, Eq. 7 value, operator
// symmetry / row sums, CG vs dense Cholesky, momentum conservation, hydrostatic
// rho*g*h; NEXT rows: Dn/Dt (dilation closed form, brute force, finite difference of the density),
// HS/ECS worked example, HL shell sum and dense solve, 2D constants and closed forms, Eq. 4 shell
// sums, list reuse against brute force on the stored sets, smoothed density at a flat interface and
// the multi-density term by brute force; pair viscosity at a two-viscosity interface (hand shell sum, brute
// force with walls), p-hat and gradient variants 0-2 by brute force with dummies carrying a pressure, the Morton
// key table, preconditioned CG against the dense solve, and -- whole steps -- the paper's water drop on both
// pressure routes (a b = R^2 and the analytic doubling time; Table 1).  The VALUES of PPE pressures
// in a moving fluid: the paper prints none => "parity unpinned" against the paper for those (pinned on the
// parts and through the water drop).
#include <algorithm>
#include <cmath>
#include <cstdint>
#include <cstring>
#include <vector>

namespace {

enum { FLUID = 0, WALL = 1, DUMMY = 2, GHOST = 3 };

struct Prm {
  int dim;
  double l0, re_n, re_lap, dt, g[3];
  int n_phases;
  double rho[2], nu[2], c0, gamma, beta, compress, ppe_relax, cg_rtol;
  int cg_maxit;
  double cs;
  int grad_variant, clamp_negative_p, rho_pair_mean, nu_pair_mean, cell_div;
  int ppe_source;     // 0: Eq. 8; 1: higher-order source Eq. 15 (HS); 2: HS + error-compensating parts Eq. 17-18 (ECS)
  int ppe_laplacian;  // 0: Eq. 10 form (Listing 2); 1: higher-order Laplacian Eq. 16 (HL)
  int kernel;         // 0: w = re/r - 1 (Eq. 3); 1: w = (1 - r/re)^3 (Eq. 4)
  int rebin_every;    // 1: exact sets at every sweep (Q7); K > 1: the paper's list reuse (Q24)
  int key_mode;       // 0: linear x-fastest cell key; 1: Morton key, 3 x 10-bit interleave (north_star "Morton- or cell-sorted")
  int cg_warm_start;  // 0: x0 = 0 (Q15); 1: x0 = the particle's previous pressure
  double dmin[3], dmax[3];
  int max_neighbours;
  double n0_n, n0_lap, lam;
};

// I2 (Eq.5 on the initial lattice; "weighted average of
// r_ij^2"): sums over the ideal cubic lattice, o in Z^dim \ {0}, |o| l0 < re.
// P:123 Eq.3 (kernel 0) and P:128 Eq.4 (kernel 1), for 0 <= r < re.
double kernel_w(int kernel, double re, double r) {
  if (kernel == 1) { const double t = 1.0 - r / re; return t * t * t; }
  return re / r - 1.0;
}

void lattice_constants(int dim, double l0, double re, double* n0, double* lam, int* count, int kernel = 0) {
  int R = (int)std::ceil(re / l0) + 1;
  double sw = 0.0, sr2w = 0.0;
  int cnt = 0;
  for (int oz = (dim == 3 ? -R : 0); oz <= (dim == 3 ? R : 0); ++oz)
    for (int oy = -R; oy <= R; ++oy)
      for (int ox = -R; ox <= R; ++ox) {
        if (ox == 0 && oy == 0 && oz == 0) continue;
        double dx = ox * l0, dy = oy * l0, dz = oz * l0;
        double r2 = (dx * dx + dy * dy) + dz * dz;
        if (r2 < re * re) {
          double r = std::sqrt(r2);
          double w = kernel_w(kernel, re, r);  // P:123 Eq.3 / P:128 Eq.4
          sw += w;
          sr2w += r2 * w;
          ++cnt;
        }
      }
  *n0 = sw;
  *lam = sr2w / sw;
  *count = cnt;
}

struct Orc {
  Prm prm;
  int n = 0;
  std::vector<double> f[22];  // x y z u v w n p ax ay az nut b phat gx gy gz xcg dndt n_k dndt_k rho_s
  std::vector<int> type, phase, bc, key, perm, cell_start;
  double h = 0, inv_h = 0;
  int nc[3] = {0, 0, 0};
  int ncells = 0;       // size of the key space: n_x n_y n_z (linear) or 8^bits (Morton)
  std::vector<int> ccx, ccy, ccz;  // cell coordinates of every particle (last BIN)
  bool brute = false;
  bool binned = false;
  double n0_n = 0, n0_lap = 0, lam = 0, A_lap = 0;
  int cg_iters = 0;
  double cg_relres = 0;
  int n_ghost = 0, n_surface = 0, max_nb = 0;

  std::vector<double>&X() { return f[0]; }
  std::vector<double>&Y() { return f[1]; }
  std::vector<double>&Z() { return f[2]; }

  void init_constants() {
    int c;
    double lam_n;
    // I1-I3
    if (prm.n0_n > 0) n0_n = prm.n0_n; else lattice_constants(prm.dim, prm.l0, prm.re_n, &n0_n, &lam_n, &c, prm.kernel);
    double n0l, lm;
    lattice_constants(prm.dim, prm.l0, prm.re_lap, &n0l, &lm, &c, prm.kernel);
    n0_lap = prm.n0_lap > 0 ? prm.n0_lap : n0l;
    lam = prm.lam > 0 ? prm.lam : lm;
    A_lap = 2.0 * prm.dim / (n0_lap * lam);  // P:170 Eq.10
    // I4 (cells "have sides equal to r_e"; cell_div = 1)
    h = std::max(prm.re_n, prm.re_lap) / prm.cell_div;
    inv_h = 1.0 / h;
    ncells = 1;
    for (int a = 0; a < 3; ++a) {
      nc[a] = (int)std::ceil((prm.dmax[a] - prm.dmin[a]) * inv_h);
      if (nc[a] < 1) nc[a] = 1;
      ncells *= nc[a];
    }
    if (prm.key_mode == 1) {  // Morton keys live in [0, 8^bits), bits = smallest with 2^bits >= every n_a
      int bits = 0;
      while ((1 << bits) < std::max(nc[0], std::max(nc[1], nc[2]))) ++bits;
      ncells = 1 << (3 * bits);
    }
  }
  // Morton key: bit k of c_x goes to bit 3k, of c_y to bit 3k+1, of c_z to bit 3k+2 (k = 0..9).
  static int morton3(int cx, int cy, int cz) {
    int key = 0;
    for (int k = 0; k < 10; ++k) {
      key |= ((cx >> k) & 1) << (3 * k);
      key |= ((cy >> k) & 1) << (3 * k + 1);
      key |= ((cz >> k) & 1) << (3 * k + 2);
    }
    return key;
  }
  int cell_key(int cx, int cy, int cz) const {
    return prm.key_mode == 1 ? morton3(cx, cy, cz) : cx + nc[0] * (cy + nc[1] * cz);
  }

  // BIN: B1-B4.
  void bin() {
    key.assign(n, 0);
    ccx.assign(n, 0); ccy.assign(n, 0); ccz.assign(n, 0);
    n_ghost = 0;
    for (int i = 0; i < n; ++i) {
      const double pos[3] = {f[0][i], f[1][i], f[2][i]};
      int c[3];
      bool out = (type[i] == GHOST);
      for (int a = 0; a < 3; ++a) {
        double fl = std::floor((pos[a] - prm.dmin[a]) * inv_h);
        if (!(fl >= 0.0 && fl < (double)nc[a])) { out = true; c[a] = 0; }
        else c[a] = (int)fl;
      }
      if (out) { type[i] = GHOST; key[i] = ncells; ++n_ghost; }  // B1, B2
      else { key[i] = cell_key(c[0], c[1], c[2]); ccx[i] = c[0]; ccy[i] = c[1]; ccz[i] = c[2]; }
    }
    // B3: stable sort by key, ties by ascending original index.
    perm.resize(n);
    for (int i = 0; i < n; ++i) perm[i] = i;
    std::stable_sort(perm.begin(), perm.end(), [&](int a, int b) { return key[a] < key[b]; });
    // B4: cell_start[c] = #{k : key[perm[k]] < c}, c = 0..ncells
    cell_start.assign(ncells + 1, 0);
    {
      int k = 0;
      for (int c = 0; c <= ncells; ++c) {
        while (k < n && key[perm[k]] < c) ++k;
        cell_start[c] = k;
      }
    }
    binned = true;
  }
  // NEXT-3 list reuse ("constant for that entire step", "every four steps"; Q24):
  // the neighbour lists of both radii as built by the last scheduled BIN, each row ascending.
  std::vector<int> lst_off[2], lst_idx[2];
  bool use_lists = false;
  long step_count = 0;
  void build_lists() {
    const double radius[2] = {prm.re_n, prm.re_lap};
    for (int w = 0; w < 2; ++w) {
      lst_off[w].assign(n + 1, 0);
      lst_idx[w].clear();
      for (int i = 0; i < n; ++i) {
        std::vector<int> row;
        for_neighbours(i, radius[w], [&](int j, double, double, double, double) { row.push_back(j); });
        std::sort(row.begin(), row.end());
        lst_idx[w].insert(lst_idx[w].end(), row.begin(), row.end());
        lst_off[w][i + 1] = (int)lst_idx[w].size();
      }
    }
  }
  void ensure_binned() { if (!use_lists && !binned) bin(); }

  // NEIGHBOURS(i, re) (Eq.3, strict r < re; Q2 rounding of the test).
  template <class F>
  void for_neighbours(int i, double re, F&& fn) {
    const double re2 = re * re;
    const double xi = f[0][i], yi = f[1][i], zi = f[2][i];
    auto test = [&](int j) {
      if (j == i || type[j] == GHOST) return;
      double dx = f[0][j] - xi, dy = f[1][j] - yi, dz = f[2][j] - zi;
      double r2 = (dx * dx + dy * dy) + dz * dz;
      if (r2 < re2) fn(j, dx, dy, dz, r2);
    };
    if (type[i] == GHOST) return;
    if (use_lists) {  // stored list of that radius, re-tested at the current distance (Q24)
      const int w = (re == prm.re_n) ? 0 : 1;
      for (int k = lst_off[w][i]; k < lst_off[w][i + 1]; ++k) test(lst_idx[w][k]);
      return;
    }
    if (brute) {
      for (int j = 0; j < n; ++j) test(j);
      return;
    }
    int R = (int)std::ceil(re * inv_h);
    int cx = ccx[i], cy = ccy[i], cz = ccz[i];
    for (int dz = -R; dz <= R; ++dz) {
      int z2 = cz + dz;
      if (z2 < 0 || z2 >= nc[2]) continue;
      for (int dy = -R; dy <= R; ++dy) {
        int y2 = cy + dy;
        if (y2 < 0 || y2 >= nc[1]) continue;
        for (int dx = -R; dx <= R; ++dx) {
          int x2 = cx + dx;
          if (x2 < 0 || x2 >= nc[0]) continue;
          int c = cell_key(x2, y2, z2);
          for (int s = cell_start[c]; s < cell_start[c + 1]; ++s) test(perm[s]);
        }
      }
    }
  }

  double w_of(double re, double r2) const { return kernel_w(prm.kernel, re, std::sqrt(r2)); }  // Eq.3 / Eq.4

  // step 6 (Eq.5): all non-ghost i; all non-ghost j count.
  void density() {
    ensure_binned();
    const double re = prm.re_n;
    max_nb = 0;
    for (int i = 0; i < n; ++i) {
      double s = 0.0;
      int cnt = 0;
      for_neighbours(i, re, [&](int, double, double, double, double r2) { s += w_of(re, r2); ++cnt; });
      f[6][i] = s;
      max_nb = std::max(max_nb, cnt);
    }
  }

  double nu_of(int i) const { return prm.nu[phase[i]] + f[11][i]; }

  // step 2 (Eq.13, [51]; Q10): Smagorinsky eddy viscosity.
  void smagorinsky() {
    ensure_binned();
    const double re = prm.re_n, d = prm.dim;
    for (int i = 0; i < n; ++i) {
      f[11][i] = 0.0;
      if (prm.cs <= 0.0 || type[i] != FLUID) continue;
      double G[3][3] = {{0, 0, 0}, {0, 0, 0}, {0, 0, 0}};  // G[a][b] = d u_b / d x_a
      const double ui[3] = {f[3][i], f[4][i], f[5][i]};
      for_neighbours(i, re, [&](int j, double dx, double dy, double dz, double r2) {
        const bool solid = (type[j] == WALL || type[j] == DUMMY);
        const double uj[3] = {solid ? 0.0 : f[3][j], solid ? 0.0 : f[4][j], solid ? 0.0 : f[5][j]};
        const double dr[3] = {dx, dy, dz};
        const double w = w_of(re, r2);
        for (int a = 0; a < 3; ++a)
          for (int b = 0; b < 3; ++b) G[a][b] += (uj[b] - ui[b]) * dr[a] / r2 * w;
      });
      double ss = 0.0;
      for (int a = 0; a < 3; ++a)
        for (int b = 0; b < 3; ++b) {
          double S = 0.5 * (d / n0_n) * (G[a][b] + G[b][a]);
          ss += S * S;
        }
      f[11][i] = (prm.cs * prm.l0) * (prm.cs * prm.l0) * std::sqrt(2.0 * ss);
    }
  }

  // step 3 (Eq.2 viscous + external term, Eq.10; Q9).
  void viscosity() {
    ensure_binned();
    smagorinsky();
    const double re = prm.re_lap;
    for (int i = 0; i < n; ++i) {
      f[8][i] = f[9][i] = f[10][i] = 0.0;
      if (type[i] != FLUID) continue;
      const double nui = nu_of(i);
      const double ui[3] = {f[3][i], f[4][i], f[5][i]};
      double s[3] = {0, 0, 0};
      for_neighbours(i, re, [&](int j, double, double, double, double r2) {
        const bool solid = (type[j] == WALL || type[j] == DUMMY);
        double nuij;
        if (solid) nuij = nui;
        else {
          const double nuj = nu_of(j);
          if (prm.nu_pair_mean == 1) nuij = (nui + nuj > 0.0) ? 2.0 * nui * nuj / (nui + nuj) : 0.0;  // Q9 (0/0 -> 0)
          else nuij = 0.5 * (nui + nuj);
        }
        const double w = w_of(re, r2);
        const double uj[3] = {solid ? 0.0 : f[3][j], solid ? 0.0 : f[4][j], solid ? 0.0 : f[5][j]};
        for (int a = 0; a < 3; ++a) s[a] += nuij * (uj[a] - ui[a]) * w;
      });
      for (int a = 0; a < 3; ++a) f[8 + a][i] = A_lap * s[a] + prm.g[a];
    }
  }

  // step 4 (Q8): explicit predictor, fluid only.
  void predict() {
    const double dt = prm.dt;
    for (int i = 0; i < n; ++i) {
      if (type[i] != FLUID) continue;
      for (int a = 0; a < 3; ++a) {
        f[3 + a][i] = f[3 + a][i] + dt * f[8 + a][i];
        f[a][i] = f[a][i] + dt * f[3 + a][i];
      }
    }
    binned = false;
  }

  // step 7a (Eq.7; Q4 clamp).
  static double eos(double rho, double c0, double gamma, double n, double n0) {
    double q = n / n0, qg;
    if (gamma == 7.0) { double q2 = q * q, q4 = q2 * q2; qg = q4 * q2 * q; }
    else qg = std::pow(q, gamma);
    return rho * c0 * c0 / gamma * (qg - 1.0);
  }
  void pressure_explicit() {
    for (int i = 0; i < n; ++i) {
      double p = 0.0;
      if (type[i] == FLUID || type[i] == WALL) {
        p = eos(prm.rho[phase[i]], prm.c0, prm.gamma, f[6][i], n0_n);
        if (prm.clamp_negative_p && p < 0.0) p = 0.0;
      }
      f[7][i] = p;
    }
  }

  // step 7b.1 (Eq.6; Listing 2 comments).
  void ppe_flags() {
    n_surface = 0;
    for (int i = 0; i < n; ++i) {
      if (type[i] == DUMMY || type[i] == GHOST) bc[i] = -1;
      else if (f[6][i] < prm.beta * n0_n) { bc[i] = 1; ++n_surface; }
      else bc[i] = 0;
    }
  }
  // NEXT-1, MPS-HS (Eq.15; Q22): the material derivative of the particle
  // number density of Eq.5 with w = re/r - 1:  Dn/Dt = sum dw/dt = - sum re/r^3 (x_ij . u_ij),
  // x_ij = x_j - x_i, u_ij = u_j - u_i (walls and dummies have u = 0), over N(i, r_n),
  // every non-ghost i.  Written into field `dst` (18: current, 20: the copy kept from r^k).
  void dndt(int dst) {
    ensure_binned();
    const double re = prm.re_n;
    for (int i = 0; i < n; ++i) {
      f[dst][i] = 0.0;
      if (type[i] == GHOST) continue;
      const bool si = (type[i] == WALL || type[i] == DUMMY);
      const double ui[3] = {si ? 0.0 : f[3][i], si ? 0.0 : f[4][i], si ? 0.0 : f[5][i]};
      double s = 0.0;
      for_neighbours(i, re, [&](int j, double dx, double dy, double dz, double r2) {
        const bool sj = (type[j] == WALL || type[j] == DUMMY);
        const double uj[3] = {sj ? 0.0 : f[3][j], sj ? 0.0 : f[4][j], sj ? 0.0 : f[5][j]};
        const double r = std::sqrt(r2);
        s += re / (r2 * r) * (dx * (uj[0] - ui[0]) + dy * (uj[1] - ui[1]) + dz * (uj[2] - ui[2]));
      });
      f[dst][i] = -s;
    }
  }
  // step 7b.2.  ppe_source 0: Eq.8 divided by -rho (Q5).
  // ppe_source 1 (HS, Eq.15; Q22): b = relax / (n0 dt) (Dn/Dt)*.
  // ppe_source 2 (ECS, Eq.17-18; Q22): b = relax / dt [ (Dn/Dt)* / n0 + ECS ],
  //   ECS = |alpha| (Dn/Dt)^k / n0 + |beta| alpha / dt, alpha = (n^k - n0)/n0,
  //   beta = dt (Dn/Dt)^k / n0, with n^k and (Dn/Dt)^k kept from the start of the step.
  void ppe_rhs() {
    const double dt = prm.dt;
    for (int i = 0; i < n; ++i) {
      double b = 0.0;
      if (bc[i] == 0) {
        if (prm.ppe_source == 0) {
          b = prm.ppe_relax / (dt * dt) * (f[6][i] - n0_n) / n0_n;
        } else if (prm.ppe_source == 1) {
          b = prm.ppe_relax / (n0_n * dt) * f[18][i];
        } else {
          const double alpha = (f[19][i] - n0_n) / n0_n;
          const double beta = dt / n0_n * f[20][i];
          const double ecs = std::fabs(alpha) * (f[20][i] / n0_n) + std::fabs(beta) * (alpha / dt);
          b = prm.ppe_relax / dt * (f[18][i] / n0_n + ecs);
        }
      }
      f[12][i] = b;
    }
  }
  // pair coefficient of the pressure Laplacian before the 1/rho_ij: Eq.10 form
  // A_lap w(r) (Listing 2), or MPS-HL (Eq.16; Q23): 2 re / (n0 r^3).
  double lap_coef(double re, double r2) const {
    if (prm.ppe_laplacian == 1) return 2.0 * re / (n0_lap * r2 * std::sqrt(r2));
    return A_lap * w_of(re, r2);
  }
  double rho_pair(int i, int j) const {
    const double ri = prm.rho[phase[i]], rj = prm.rho[phase[j]];
    return prm.rho_pair_mean == 1 ? 2.0 * ri * rj / (ri + rj) : 0.5 * (ri + rj);  // Q6
  }
  // step 7b.3 (Listing 2: off-diagonal -val, diagonal += val, diagonal
  // += 1.00e-7/dt^2, dummy neighbours give 0, rows only where bcon == 0).
  // Positions are fixed during a solve, so ppe_solve() records, for every row, the neighbours and
  // r2 in the order for_neighbours() visits them and the later applications walk that record:
  // the same pairs, the same numbers, the same order of additions -- only the search is skipped
  // (this is Listing 2's neigh[] list).
  std::vector<long long> nbc_off;
  std::vector<int> nbc_j;
  std::vector<double> nbc_r2;
  bool nbc_on = false;
  void nbc_build() {
    const double re = prm.re_lap;
    nbc_off.assign(n + 1, 0);
    nbc_j.clear();
    nbc_r2.clear();
    for (int i = 0; i < n; ++i) {
      if (bc[i] == 0)
        for_neighbours(i, re, [&](int j, double, double, double, double r2) { nbc_j.push_back(j); nbc_r2.push_back(r2); });
      nbc_off[i + 1] = (long long)nbc_j.size();
    }
    nbc_on = true;
  }
  void nbc_drop() { nbc_on = false; nbc_off.clear(); nbc_j.clear(); nbc_r2.clear(); nbc_j.shrink_to_fit(); nbc_r2.shrink_to_fit(); }
  template <class F>
  void for_lap_neighbours(int i, F&& fn) {
    if (nbc_on) { for (long long k = nbc_off[i]; k < nbc_off[i + 1]; ++k) fn(nbc_j[k], nbc_r2[k]); }
    else for_neighbours(i, prm.re_lap, [&](int j, double, double, double, double r2) { fn(j, r2); });
  }
  void ppe_apply(const double* xin, double* yout) {
    ensure_binned();
    const double re = prm.re_lap;
    for (int i = 0; i < n; ++i) {
      yout[i] = 0.0;
      if (bc[i] != 0) continue;
      double s = 0.0;
      const double xi = xin[i];
      for_lap_neighbours(i, [&](int j, double r2) {
        if (bc[j] == -1) return;
        const double c = lap_coef(re, r2) / rho_pair(i, j);
        s += c * (xi - (bc[j] == 0 ? xin[j] : 0.0));
      });
      yout[i] = s + prm.compress / (prm.dt * prm.dt) * xi;
    }
  }
  // step 7b.4 (Eq.9, P:176 CG part; Q15): textbook CG, x0 = 0 (or, cg_warm_start = 1, the
  // particle's previous pressure on the rows: r0 = b - A x0).
  bool nbc_keep = false;  // set by the preconditioned solvers, which build the record themselves
  int ppe_solve(double rtol, int maxit) {
    std::vector<double>& x = f[17];
    std::vector<double> r(n), p(n), Ap(n);
    const std::vector<double>& b = f[12];
    double rr = 0.0, bb = 0.0;
    ensure_binned();
    nbc_build();
    for (int i = 0; i < n; ++i) { x[i] = 0.0; r[i] = b[i]; }
    if (prm.cg_warm_start) {
      for (int i = 0; i < n; ++i) x[i] = (bc[i] == 0) ? f[7][i] : 0.0;
      ppe_apply(x.data(), Ap.data());
      for (int i = 0; i < n; ++i) r[i] = (bc[i] == 0) ? b[i] - Ap[i] : 0.0;
    }
    for (int i = 0; i < n; ++i) p[i] = r[i];
    for (int i = 0; i < n; ++i) if (bc[i] == 0) { rr += r[i] * r[i]; bb += b[i] * b[i]; }
    cg_iters = 0;
    cg_relres = 0.0;
    if (bb == 0.0) { for (int i = 0; i < n; ++i) x[i] = 0.0; nbc_drop(); return 0; }
    if (rr <= rtol * rtol * bb) { cg_relres = std::sqrt(rr / bb); nbc_drop(); return 0; }
    int it;
    bool conv = false;
    for (it = 1; it <= maxit; ++it) {
      ppe_apply(p.data(), Ap.data());
      double pAp = 0.0;
      for (int i = 0; i < n; ++i) if (bc[i] == 0) pAp += p[i] * Ap[i];
      const double alpha = rr / pAp;
      double rr2 = 0.0;
      for (int i = 0; i < n; ++i) if (bc[i] == 0) {
        x[i] += alpha * p[i];
        r[i] -= alpha * Ap[i];
        rr2 += r[i] * r[i];
      }
      if (rr2 <= rtol * rtol * bb) { rr = rr2; conv = true; break; }
      const double beta = rr2 / rr;
      for (int i = 0; i < n; ++i) if (bc[i] == 0) p[i] = r[i] + beta * p[i];
      rr = rr2;
    }
    cg_iters = conv ? it : maxit;
    cg_relres = std::sqrt(rr / bb);
    nbc_drop();
    return conv ? cg_iters : -cg_iters;
  }

  // ---- NEXT-4 ("incomplete Cholesky conjugate gradient"): preconditioned CG ------------
  // The rows bc = 0 of Listing 2's matrix written out as CSR in the order of the
  // cell-sorted slots (perm): diagonal = sum of c_ij over non-dummy neighbours + compress/dt^2,
  // off-diagonal -c_ij where j is an unknown too.  precond: 0 none, 1 Jacobi (diagonal),
  // 2 block Jacobi with the grid cells as blocks (dense Cholesky of each block), 3 incomplete Cholesky
  // with zero fill-in IC(0) (the paper's ICCG), 4 Chebyshev polynomial of degree `degree` on
  // [lmax / ratio, lmax].  Textbook PCG (Saad, Alg. 9.1) from x0 = 0; the stopping rule is the
  // oracle's: ||r|| <= rtol ||b|| on the unpreconditioned residual.
  struct Csr { int m = 0; std::vector<int> off, col; std::vector<double> val, diag; std::vector<int> row_of, slot; };
  Csr pcg_assemble() {
    Csr A;
    ensure_binned();
    const double re = prm.re_lap;
    A.row_of.assign(n, -1);
    for (int s = 0; s < n; ++s) { int i = perm[s]; if (bc[i] == 0) { A.row_of[i] = A.m++; A.slot.push_back(i); } }
    A.off.assign(A.m + 1, 0); A.diag.assign(A.m, 0.0);
    for (int r = 0; r < A.m; ++r) {
      const int i = A.slot[r];
      std::vector<std::pair<int, double>> ent;
      double d = prm.compress / (prm.dt * prm.dt);
      for_neighbours(i, re, [&](int j, double, double, double, double r2) {
        if (bc[j] == -1) return;
        const double c = lap_coef(re, r2) / rho_pair(i, j);
        d += c;
        if (bc[j] == 0) ent.push_back({A.row_of[j], -c});
      });
      std::sort(ent.begin(), ent.end());
      for (auto& e : ent) { A.col.push_back(e.first); A.val.push_back(e.second); }
      A.diag[r] = d;
      A.off[r + 1] = (int)A.col.size();
    }
    return A;
  }
  static void csr_apply(const Csr& A, const std::vector<double>& x, std::vector<double>& y) {
    for (int r = 0; r < A.m; ++r) {
      double s = A.diag[r] * x[r];
      for (int k = A.off[r]; k < A.off[r + 1]; ++k) s += A.val[k] * x[A.col[k]];
      y[r] = s;
    }
  }
  int pcg_iters = 0;
  double pcg_relres = 0.0;
  int ppe_solve_pcg(double rtol, int maxit, int precond, int degree, double ratio) {
    Csr A = pcg_assemble();
    const int m = A.m;
    std::vector<double> b(m), x(m, 0.0), r(m), z(m), p(m), Ap(m);
    for (int q = 0; q < m; ++q) b[q] = f[12][A.slot[q]];
    // --- set-up of M
    std::vector<double> Ld;                 // IC(0): diagonal of L; lower part shares A's pattern
    std::vector<double> Lv;
    std::vector<int> blk_of, blk_off, blk_rows;  // block Jacobi
    std::vector<std::vector<double>> blkL;
    double lmax = 0.0;
    if (precond == 3) {
      Lv = A.val; Ld = A.diag;
      // row-oriented IC(0): for row r, for each lower entry (r, k): L_rk = (a_rk - sum_{j<k} L_rj L_kj) / L_kk
      for (int r2 = 0; r2 < m; ++r2) {
        for (int a = A.off[r2]; a < A.off[r2 + 1] && A.col[a] < r2; ++a) {
          const int k = A.col[a];
          double sum = Lv[a];
          int pa = A.off[r2], pb = A.off[k];
          while (pa < a && pb < A.off[k + 1] && A.col[pb] < k) {
            if (A.col[pa] == A.col[pb]) { sum -= Lv[pa] * Lv[pb]; ++pa; ++pb; }
            else if (A.col[pa] < A.col[pb]) ++pa; else ++pb;
          }
          Lv[a] = sum / Ld[k];
        }
        double d = A.diag[r2];
        for (int a = A.off[r2]; a < A.off[r2 + 1] && A.col[a] < r2; ++a) d -= Lv[a] * Lv[a];
        if (!(d > 0.0)) return -1000000;  // breakdown (cannot happen for this M-matrix)
        Ld[r2] = std::sqrt(d);
      }
    } else if (precond == 2) {
      // blocks = grid cells (rows are in cell-sorted order, so a block is a run of consecutive rows)
      blk_of.assign(m, 0);
      int nb = 0, last = -1;
      for (int q = 0; q < m; ++q) { int kq = key[A.slot[q]]; if (kq != last) { blk_off.push_back(q); last = kq; ++nb; } blk_of[q] = nb - 1; }
      blk_off.push_back(m);
      blkL.resize(nb);
      for (int bq = 0; bq < nb; ++bq) {
        const int lo = blk_off[bq], sz = blk_off[bq + 1] - lo;
        std::vector<double>& M = blkL[bq];
        M.assign((size_t)sz * sz, 0.0);
        for (int q = 0; q < sz; ++q) {
          M[(size_t)q * sz + q] = A.diag[lo + q];
          for (int k = A.off[lo + q]; k < A.off[lo + q + 1]; ++k) {
            const int c2 = A.col[k] - lo;
            if (c2 >= 0 && c2 < sz) M[(size_t)q * sz + c2] = A.val[k];
          }
        }
        for (int j = 0; j < sz; ++j) {       // dense Cholesky, lower triangle in place
          double d = M[(size_t)j * sz + j];
          for (int k = 0; k < j; ++k) d -= M[(size_t)j * sz + k] * M[(size_t)j * sz + k];
          d = std::sqrt(d);
          M[(size_t)j * sz + j] = d;
          for (int i2 = j + 1; i2 < sz; ++i2) {
            double v = M[(size_t)i2 * sz + j];
            for (int k = 0; k < j; ++k) v -= M[(size_t)i2 * sz + k] * M[(size_t)j * sz + k];
            M[(size_t)i2 * sz + j] = v / d;
          }
        }
      }
    } else if (precond == 4) {
      for (int q = 0; q < m; ++q) {          // Gershgorin bound of the largest eigenvalue
        double s2 = A.diag[q];
        for (int k = A.off[q]; k < A.off[q + 1]; ++k) s2 += std::fabs(A.val[k]);
        lmax = std::max(lmax, s2);
      }
    }
    auto apply_M = [&](const std::vector<double>& rin, std::vector<double>& zout) {
      if (precond == 1) { for (int q = 0; q < m; ++q) zout[q] = rin[q] / A.diag[q]; }
      else if (precond == 2) {
        for (size_t bq = 0; bq + 1 < blk_off.size(); ++bq) {
          const int lo = blk_off[bq], sz = blk_off[bq + 1] - lo;
          const std::vector<double>& M = blkL[bq];
          for (int i2 = 0; i2 < sz; ++i2) { double v = rin[lo + i2]; for (int k = 0; k < i2; ++k) v -= M[(size_t)i2 * sz + k] * zout[lo + k]; zout[lo + i2] = v / M[(size_t)i2 * sz + i2]; }
          for (int i2 = sz - 1; i2 >= 0; --i2) { double v = zout[lo + i2]; for (int k = i2 + 1; k < sz; ++k) v -= M[(size_t)k * sz + i2] * zout[lo + k]; zout[lo + i2] = v / M[(size_t)i2 * sz + i2]; }
        }
      } else if (precond == 3) {
        // L y = r (forward), L^T z = y (backward, column-oriented)
        for (int q = 0; q < m; ++q) {
          double v = rin[q];
          for (int a = A.off[q]; a < A.off[q + 1] && A.col[a] < q; ++a) v -= Lv[a] * zout[A.col[a]];
          zout[q] = v / Ld[q];
        }
        for (int q = m - 1; q >= 0; --q) {
          zout[q] /= Ld[q];
          const double zq = zout[q];
          for (int a = A.off[q]; a < A.off[q + 1] && A.col[a] < q; ++a) zout[A.col[a]] -= Lv[a] * zq;
        }
      } else if (precond == 4) {
        // `degree` steps of the Chebyshev iteration for A z = r from z = 0 on [lmax/ratio, lmax]
        const double lmin = lmax / ratio, theta = 0.5 * (lmax + lmin), delta = 0.5 * (lmax - lmin);
        std::vector<double> res(rin), d(m), t(m);
        double sigma = theta / delta, rho_c = 1.0 / sigma;
        for (int q = 0; q < m; ++q) { d[q] = res[q] / theta; zout[q] = 0.0; }
        for (int it = 0; it < degree; ++it) {
          for (int q = 0; q < m; ++q) zout[q] += d[q];
          if (it + 1 == degree) break;
          csr_apply(A, d, t);
          for (int q = 0; q < m; ++q) res[q] -= t[q];
          const double rho_n = 1.0 / (2.0 * sigma - rho_c);
          for (int q = 0; q < m; ++q) d[q] = rho_n * rho_c * d[q] + 2.0 * rho_n / delta * res[q];
          rho_c = rho_n;
        }
      } else zout = rin;
    };
    double bb = 0.0;
    for (int q = 0; q < m; ++q) { r[q] = b[q]; bb += b[q] * b[q]; }
    pcg_iters = 0; pcg_relres = 0.0;
    std::vector<double>& xs = f[17];
    for (int i = 0; i < n; ++i) xs[i] = 0.0;
    if (bb == 0.0) return 0;
    apply_M(r, z);
    p = z;
    double rz = 0.0;
    for (int q = 0; q < m; ++q) rz += r[q] * z[q];
    int it; bool conv = false; double rr = bb;
    for (it = 1; it <= maxit; ++it) {
      csr_apply(A, p, Ap);
      double pAp = 0.0;
      for (int q = 0; q < m; ++q) pAp += p[q] * Ap[q];
      const double alpha = rz / pAp;
      rr = 0.0;
      for (int q = 0; q < m; ++q) { x[q] += alpha * p[q]; r[q] -= alpha * Ap[q]; rr += r[q] * r[q]; }
      if (rr <= rtol * rtol * bb) { conv = true; break; }
      apply_M(r, z);
      double rz2 = 0.0;
      for (int q = 0; q < m; ++q) rz2 += r[q] * z[q];
      const double beta = rz2 / rz;
      for (int q = 0; q < m; ++q) p[q] = z[q] + beta * p[q];
      rz = rz2;
    }
    pcg_iters = conv ? it : maxit;
    pcg_relres = std::sqrt(rr / bb);
    for (int q = 0; q < m; ++q) xs[A.slot[q]] = x[q];
    return conv ? pcg_iters : -pcg_iters;
  }

  // step 7b (whole) incl. 7b.5 (Q4 clamp).
  int pressure_ppe() {
    ppe_flags();
    ppe_rhs();
    int it = ppe_solve(prm.cg_rtol, prm.cg_maxit);
    for (int i = 0; i < n; ++i) {
      double p = (bc[i] == 0) ? f[17][i] : 0.0;
      if (prm.clamp_negative_p && p < 0.0) p = 0.0;
      f[7][i] = p;
    }
    return it;
  }

  // step 8 (P:215 phi-hat of Eq.14; Q12).
  void phat() {
    ensure_binned();
    const double re = prm.re_n;
    for (int i = 0; i < n; ++i) {
      f[13][i] = 0.0;
      if (type[i] != FLUID && type[i] != WALL) continue;
      double m = f[7][i];
      for_neighbours(i, re, [&](int j, double, double, double, double) {
        if (type[j] == DUMMY) return;
        if (f[7][j] < m) m = f[7][j];
      });
      f[13][i] = m;
    }
  }
  // NEXT-2 (Q25): the smoothed density <rho>_i "set for each particle before starting
  // the simulation": kernel-weighted mean of the neighbours' densities over N(i, r_n).
  bool rho_s_ready = false;
  void smooth_density() {
    ensure_binned();
    const double re = prm.re_n;
    for (int i = 0; i < n; ++i) {
      double sw = 0.0, srw = 0.0;
      for_neighbours(i, re, [&](int j, double, double, double, double r2) {
        const double w = w_of(re, r2);
        sw += w;
        srw += prm.rho[phase[j]] * w;
      });
      f[21][i] = sw > 0.0 ? srw / sw : prm.rho[phase[i]];
    }
    rho_s_ready = true;
  }
  // step 9, variant 3 (Eq.11-12; Q25): the multi-density pressure term of the
  // weakly-compressible model, alpha_i = p_i / rho_i (Eq.12 times nothing: p_i = rho_i alpha_i),
  //   (1/rho_i) <grad p>_i = (d/n0) sum ((<rho>_j / <rho>_i) alpha_j - alpha_i) / r^2 r_ij w,
  // stored as G_i = rho_i x that, so that the corrector's (dt / rho_i) G_i applies it as is.
  void gradient_multiphase() {
    ensure_binned();
    const double re = prm.re_n, d = prm.dim;
    for (int i = 0; i < n; ++i) {
      f[14][i] = f[15][i] = f[16][i] = 0.0;
      if (type[i] != FLUID) continue;
      const double rho_i = prm.rho[phase[i]];
      const double ai = f[7][i] / rho_i, rsi = f[21][i];
      double s[3] = {0, 0, 0};
      for_neighbours(i, re, [&](int j, double dx, double dy, double dz, double r2) {
        if (type[j] == DUMMY) return;
        const double aj = f[7][j] / prm.rho[phase[j]];
        const double c = (f[21][j] / rsi * aj - ai) / r2 * w_of(re, r2);
        s[0] += c * dx; s[1] += c * dy; s[2] += c * dz;
      });
      for (int a = 0; a < 3; ++a) f[14 + a][i] = rho_i * (d / n0_n * s[a]);
    }
  }
  // step 9 (variant 0: cited method [8], BASELINE cfg 2; variant 1: Eq.14
  // as printed; variant 2: BASELINE cfg 3 wording "(P_i+P_j)/r^2"; Q13).
  void gradient() {
    if (prm.grad_variant == 3) { gradient_multiphase(); return; }
    ensure_binned();
    const double re = prm.re_n, d = prm.dim;
    for (int i = 0; i < n; ++i) {
      f[14][i] = f[15][i] = f[16][i] = 0.0;
      if (type[i] != FLUID) continue;
      double s[3] = {0, 0, 0};
      const double pi = f[7][i], phi = f[13][i];
      for_neighbours(i, re, [&](int j, double dx, double dy, double dz, double r2) {
        if (type[j] == DUMMY) return;
        double coef;
        if (prm.grad_variant == 0) coef = f[7][j] - phi;
        else if (prm.grad_variant == 1) coef = (pi + f[7][j]) - (phi + f[13][j]);
        else coef = pi + f[7][j];
        const double c = coef / r2 * w_of(re, r2);
        s[0] += c * dx; s[1] += c * dy; s[2] += c * dz;
      });
      for (int a = 0; a < 3; ++a) f[14 + a][i] = d / n0_n * s[a];
    }
  }
  // step 10 ("first-order Euler integration"; Q8, Q3, Q11).
  void correct() {
    const double dt = prm.dt;
    for (int i = 0; i < n; ++i) {
      if (type[i] != FLUID) continue;
      const double rho = prm.rho[phase[i]];
      for (int a = 0; a < 3; ++a) {
        const double us = f[3 + a][i];
        const double un = us - dt / rho * f[14 + a][i];
        f[3 + a][i] = un;
        f[a][i] = f[a][i] + dt * (un - us);
      }
    }
    binned = false;
  }
  // STEP with list reuse (Q24): BIN and the lists of both radii only when step_count is a
  // multiple of rebin_every, at r^k; every sweep of this and the next rebin_every - 1 steps walks
  // those lists and keeps the pairs whose CURRENT distance is below the radius.
  int step_reuse(int route) {
    if (step_count % prm.rebin_every == 0) {
      use_lists = false;
      bin();
      if (prm.grad_variant == 3 && !rho_s_ready) smooth_density();
      build_lists();
    }
    use_lists = true;
    if (route == 1 && prm.ppe_source == 2) {
      density();
      f[19] = f[6];
      dndt(20);
    }
    viscosity();
    predict();
    density();
    if (route == 1 && prm.ppe_source >= 1) dndt(18);
    int rc = 0;
    if (route == 0) pressure_explicit();
    else rc = pressure_ppe();
    phat();
    gradient();
    correct();
    ++step_count;
    return rc;
  }
  // STEP k -> k+1 (section 8(c).1 of SURVEY.md / DESIGN.md section 2).
  int step(int route) {
    if (prm.rebin_every > 1) return step_reuse(route);
    bin();                // 1
    if (prm.grad_variant == 3 && !rho_s_ready) smooth_density();  // once, at the initial positions
    if (route == 1 && prm.ppe_source == 2) {  // ECS keeps n^k and (Dn/Dt)^k (Eq.17)
      density();
      f[19] = f[6];
      dndt(20);
    }
    viscosity();          // 2, 3
    predict();            // 4
    bin();                // 5
    density();            // 6
    if (route == 1 && prm.ppe_source >= 1) dndt(18);  // (Dn/Dt)* at r*, u* (Eq.15)
    int rc = 0;
    if (route == 0) pressure_explicit();  // 7a
    else rc = pressure_ppe();             // 7b
    phat();               // 8
    gradient();           // 9
    correct();            // 10
    return rc;
  }
};

}  // namespace

// ---------------------------------------------------------------------------
// C interface (loaded with ctypes by oracle/mps_oracle.py).
// dp / ip: flat parameter arrays, order fixed in oracle/mps_oracle.py.
// ---------------------------------------------------------------------------
extern "C" {

void* orc_create(const double* dp, const int* ip, int n, const double* x, const double* y,
                 const double* z, const double* u, const double* v, const double* w,
                 const int* type, const int* phase) {
  Orc* o = new Orc;
  Prm& p = o->prm;
  p.l0 = dp[0]; p.re_n = dp[1]; p.re_lap = dp[2]; p.dt = dp[3];
  p.g[0] = dp[4]; p.g[1] = dp[5]; p.g[2] = dp[6];
  p.rho[0] = dp[7]; p.rho[1] = dp[8]; p.nu[0] = dp[9]; p.nu[1] = dp[10];
  p.c0 = dp[11]; p.gamma = dp[12]; p.beta = dp[13]; p.compress = dp[14];
  p.ppe_relax = dp[15]; p.cg_rtol = dp[16]; p.cs = dp[17];
  for (int a = 0; a < 3; ++a) { p.dmin[a] = dp[18 + a]; p.dmax[a] = dp[21 + a]; }
  p.n0_n = dp[24]; p.n0_lap = dp[25]; p.lam = dp[26];
  p.dim = ip[0]; p.n_phases = ip[1]; p.cg_maxit = ip[2]; p.grad_variant = ip[3];
  p.clamp_negative_p = ip[4]; p.rho_pair_mean = ip[5]; p.nu_pair_mean = ip[6];
  p.cell_div = ip[7]; p.max_neighbours = ip[8]; p.ppe_source = ip[9]; p.ppe_laplacian = ip[10]; p.kernel = ip[11]; p.rebin_every = ip[12] < 1 ? 1 : ip[12];
  p.key_mode = ip[13]; p.cg_warm_start = ip[14];
  o->n = n;
  for (auto& a : o->f) a.assign(n, 0.0);
  const double* src[6] = {x, y, z, u, v, w};
  for (int k = 0; k < 6; ++k) std::copy(src[k], src[k] + n, o->f[k].begin());
  o->type.assign(type, type + n);
  o->phase.assign(phase, phase + n);
  o->bc.assign(n, 0);
  o->init_constants();
  return o;
}
void orc_destroy(void* h) { delete (Orc*)h; }
void orc_set_brute(void* h, int b) { ((Orc*)h)->brute = (b != 0); }

int orc_set_f64(void* h, int field, const double* src) {
  Orc* o = (Orc*)h;
  if (field < 0 || field >= 22) return -1;
  std::copy(src, src + o->n, o->f[field].begin());
  if (field < 3) o->binned = false;
  if (field == 21) o->rho_s_ready = true;
  return 0;
}
int orc_get_f64(void* h, int field, double* dst) {
  Orc* o = (Orc*)h;
  if (field < 0 || field >= 22) return -1;
  std::copy(o->f[field].begin(), o->f[field].end(), dst);
  return 0;
}
static std::vector<int>* ivec(Orc* o, int field) {
  switch (field) {
    case 0: return &o->type;
    case 1: return &o->phase;
    case 2: return &o->bc;
    case 3: return &o->key;
    case 4: return &o->perm;
  }
  return nullptr;
}
int orc_set_i32(void* h, int field, const int* src) {
  Orc* o = (Orc*)h;
  std::vector<int>* v = ivec(o, field);
  if (!v || field > 2) return -1;
  v->assign(src, src + o->n);
  if (field == 0) o->binned = false;
  return 0;
}
int orc_get_i32(void* h, int field, int* dst) {
  Orc* o = (Orc*)h;
  std::vector<int>* v = ivec(o, field);
  if (!v || (int)v->size() != o->n) return -1;
  std::copy(v->begin(), v->end(), dst);
  return 0;
}
void orc_constants(void* h, double* out) {
  Orc* o = (Orc*)h;
  out[0] = o->n0_n; out[1] = o->n0_lap; out[2] = o->lam; out[3] = o->A_lap;
  out[4] = o->h; out[5] = o->inv_h;
}
void orc_grid(void* h, int* out) {
  Orc* o = (Orc*)h;
  out[0] = o->nc[0]; out[1] = o->nc[1]; out[2] = o->nc[2]; out[3] = o->ncells;
}
void orc_stats(void* h, double* out) {
  Orc* o = (Orc*)h;
  out[0] = o->cg_iters; out[1] = o->cg_relres; out[2] = o->n_ghost;
  out[3] = o->n_surface; out[4] = o->max_nb;
}
int orc_bin(void* h) { ((Orc*)h)->bin(); return 0; }
int orc_get_cell_start(void* h, int* dst) {
  Orc* o = (Orc*)h;
  std::copy(o->cell_start.begin(), o->cell_start.end(), dst);
  return 0;
}
// Neighbour sets as CSR in original numbering, each row ascending.  idx may be
// NULL (count only).  Returns the total number of entries.
long long orc_neighbours(void* h, double re, int* counts, int* idx, long long cap) {
  Orc* o = (Orc*)h;
  o->ensure_binned();
  long long tot = 0;
  std::vector<int> row;
  for (int i = 0; i < o->n; ++i) {
    row.clear();
    o->for_neighbours(i, re, [&](int j, double, double, double, double) { row.push_back(j); });
    std::sort(row.begin(), row.end());
    counts[i] = (int)row.size();
    if (idx) for (int j : row) { if (tot < cap) idx[tot] = j; ++tot; }
    else tot += (long long)row.size();
  }
  return tot;
}
int orc_density(void* h) { ((Orc*)h)->density(); return 0; }
int orc_viscosity(void* h) { ((Orc*)h)->viscosity(); return 0; }
int orc_predict(void* h) { ((Orc*)h)->predict(); return 0; }
int orc_pressure_explicit(void* h) { ((Orc*)h)->pressure_explicit(); return 0; }
int orc_ppe_flags(void* h) { ((Orc*)h)->ppe_flags(); return 0; }
int orc_ppe_rhs(void* h) { ((Orc*)h)->ppe_rhs(); return 0; }
int orc_ppe_apply(void* h, const double* xin, double* yout) { ((Orc*)h)->ppe_apply(xin, yout); return 0; }
int orc_ppe_solve(void* h, double rtol, int maxit) { return ((Orc*)h)->ppe_solve(rtol, maxit); }
int orc_ppe_solve_pcg(void* h, double rtol, int maxit, int precond, int degree, double ratio) {
  return ((Orc*)h)->ppe_solve_pcg(rtol, maxit, precond, degree, ratio);
}
int orc_morton3(int cx, int cy, int cz) { return Orc::morton3(cx, cy, cz); }
int orc_pressure_ppe(void* h) { return ((Orc*)h)->pressure_ppe(); }
void orc_smooth_density(void* h) { ((Orc*)h)->smooth_density(); }
void orc_dndt(void* h, int dst) { ((Orc*)h)->dndt(dst == 20 ? 20 : 18); }
int orc_phat(void* h) { ((Orc*)h)->phat(); return 0; }
int orc_gradient(void* h) { ((Orc*)h)->gradient(); return 0; }
int orc_correct(void* h) { ((Orc*)h)->correct(); return 0; }
// list reuse for the tests: BIN + lists at the current positions, then walk them (1) or drop them (0)
void orc_freeze_lists(void* h, int on) {
  Orc* o = (Orc*)h;
  o->use_lists = false;
  if (on) { o->bin(); o->build_lists(); o->use_lists = true; }
}
int orc_step(void* h, int nsteps, int route) {
  int rc = 0;
  for (int s = 0; s < nsteps; ++s) rc = ((Orc*)h)->step(route);
  return rc;
}
void orc_lattice_constants_k(int dim, double l0, double re, int kernel, double* out) {
  double n0, lam;
  int c;
  lattice_constants(dim, l0, re, &n0, &lam, &c, kernel);
  out[0] = n0; out[1] = lam; out[2] = c;
}
void orc_lattice_constants(int dim, double l0, double re, double* out) {
  double n0, lam; int c;
  lattice_constants(dim, l0, re, &n0, &lam, &c);
  out[0] = n0; out[1] = lam; out[2] = c;
}
double orc_eos(double rho, double c0, double gamma, double n, double n0) {
  return Orc::eos(rho, c0, gamma, n, n0);
}

}  // extern "C"
