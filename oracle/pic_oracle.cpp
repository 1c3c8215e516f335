// ORACLE — TEST INFRASTRUCTURE, NOT THE PRODUCT.
//
// Plain, slow, serial CPU implementation of one electromagnetic PIC step
// (sort -> gather -> Boris push -> Esirkepov deposit -> Yee B/E/B update),
// written from the method's definitions. It shares no code, header, table or
// helper with the CUDA path under paper_2101_12149_b200/csrc and neither side
// includes the other. Only tests/, __graft_entry__.smoke() and bench.py's
// cpu_baseline / --impl reference legs may load this library.
//
// Authority: /root/reference/PAPER.md names the steps (fused gather+push
// PAPER.md:114 §3.1; Esirkepov deposition PAPER.md:167-175 §3.4.1, ref [8]
// PAPER.md:301; counting sort by cell PAPER.md:185-203 §3.4.2; Yee staggering
// "B on faces, E and J on edges" PAPER.md:78 §2.4, ref [28] PAPER.md:323) but
// prints none of the formulas. The formulas are the textbook definitions the
// paper cites, in the reading fixed by SURVEY.md §8(c) and listed in DESIGN.md
// ("Readings"). Every function below names the step of that reading it follows.
//
// Parity pins (tests/test_oracle_*.py, all -m "not gpu"): shape partition of
// unity and first moment (T1), Boris gyration angle/radius (T2), hyperbolic
// motion (T3), Yee numerical dispersion (T4), Esirkepov continuity (T5), first
// moment of J (T6), brute-force dense deposit (T7), Gauss-law constancy (T8),
// plasma oscillation (T9), stable sort vs numpy (T10), order independence (T11), the OpenMP variant against
// the serial oracle (T12), Vay (T13), Galerkin gather (T14), CKC (T15), step 2f / diagnostics / truncated-axis
// field reads (tests/test_oracle_pins_boundaries.py). Nothing here is "parity unpinned".
//
// Build: g++ -O2 -ffp-contract=off -fopenmp -shared -fPIC (no FMA contraction, so the
// integer cell rule below is one rounded multiply exactly as written).

#include <omp.h>

#include <cmath>
#include <cstdint>
#include <cstring>
#include <vector>
#include <algorithm>
#include <string>

namespace {

// CODATA 2018. The CUDA side carries its own copy.
constexpr double kC    = 299792458.0;
constexpr double kEps0 = 8.8541878128e-12;

// Yee staggering: offset of each component from the node, in cells.
// comp 0..2 = Ex,Ey,Ez (edges; J the same), 3..5 = Bx,By,Bz (faces).
const double kStag[6][3] = {
  {0.5, 0.0, 0.0}, {0.0, 0.5, 0.0}, {0.0, 0.0, 0.5},
  {0.0, 0.5, 0.5}, {0.5, 0.0, 0.5}, {0.5, 0.5, 0.0}};

// ---------------------------------------------------------------- step 2a
// Shape factors of order n at normalised coordinate xi: leftmost index l and
// n+1 weights (B-splines of order 1..3).
template <class R>
void shape(int n, R xi, int* l, R* w) {
  if (n == 0) {                         // nearest grid point (only the Galerkin gather at order 1 uses it)
    R m = std::floor(xi + R(0.5));
    *l = (int)m;
    w[0] = R(1);
  } else if (n == 1) {
    R m = std::floor(xi);
    R d = xi - m;
    *l = (int)m;
    w[0] = R(1) - d;
    w[1] = d;
  } else if (n == 2) {
    R m = std::floor(xi + R(0.5));
    R d = xi - m;                       // in [-1/2, 1/2)
    *l = (int)m - 1;
    w[0] = R(0.5) * (R(0.5) - d) * (R(0.5) - d);
    w[1] = R(0.75) - d * d;
    w[2] = R(0.5) * (R(0.5) + d) * (R(0.5) + d);
  } else {
    R m = std::floor(xi);
    R d = xi - m;
    R e = R(1) - d;
    *l = (int)m - 1;
    w[0] = e * e * e / R(6);
    w[1] = (R(4) - R(6) * d * d + R(3) * d * d * d) / R(6);
    w[2] = (R(4) - R(6) * e * e + R(3) * e * e * e) / R(6);
    w[3] = d * d * d / R(6);
  }
}

template <class R>
struct Species {
  std::vector<R> x, y, z, ux, uy, uz, w;
  std::vector<int64_t> id;
  std::vector<int32_t> cell, perm;   // state of the most recent sort
  double q, m;
  R kq;        // q*dt/(2m)
  R jf[3];     // q/(dt*dx_a*dx_b)
};

template <class R>
struct Sim {
  int N[3];
  double dx[3], dt;
  int order;
  int periodic[3];
  int tile[3];
  int sort_interval, key_mode;
  int pusher = 0;        // 0 Boris (reading Q2), 1 Vay (ref [21])
  int solver = 0;        // 0 Yee (ref [28]), 1 CKC (Cole-Karkkainen-Cowan, ref [12])
  R ck_a[3], ck_b[3][3], ck_g[3];   // CKC: alpha_a, beta_ab (b != a), gamma_a, in working precision
  int gather_mode = 0;   // 0 uniform order (reading Q1), 1 Galerkin / energy-conserving (NEXT-2)
  // coefficient block (C-list): computed in double, rounded once to R
  R inv_dx[3], L[3], cB[3], cE[3], cJ, inv_c2, dtr;
  std::vector<R> F[6];        // Ex,Ey,Ez,Bx,By,Bz ; x fastest
  std::vector<double> Jd[3];  // J accumulated in double (reading Q10)
  std::vector<R> J[3];        // J rounded once to R before the E update
  std::vector<Species<R>> sp;
  int64_t step_count = 0;
  int64_t n_deactivated = 0;
  int omp_threads = 1;   // > 1 only inside the OpenMP variant (orc_step_omp)

  size_t ncell() const { return (size_t)N[0] * N[1] * N[2]; }

  // index rule: periodic axis -> modulo N; other axis -> out of range = -1
  // (read returns 0, write is dropped; SURVEY.md §8(c) "Grid", reading Q6)
  int wrap(int d, int i) const {
    if (periodic[d]) {
      i %= N[d];
      if (i < 0) i += N[d];
      return i;
    }
    return (i < 0 || i >= N[d]) ? -1 : i;
  }
  // linear index or -1
  int64_t lin(int i, int j, int k) const {
    i = wrap(0, i); j = wrap(1, j); k = wrap(2, k);
    if (i < 0 || j < 0 || k < 0) return -1;
    return (int64_t)i + (int64_t)N[0] * ((int64_t)j + (int64_t)N[1] * k);
  }
  R rd(const std::vector<R>& a, int i, int j, int k) const {
    int64_t t = lin(i, j, k);
    return t < 0 ? R(0) : a[(size_t)t];
  }
};

// ---------------------------------------------------------------- step 2b
// Gather one staggered component at a particle (uniform order n on every axis,
// each component interpolated from its own location; reading Q1).
template <class R>
R gather(const Sim<R>& s, int comp, R x, R y, R z) {
  int n = s.order;
  int l[3];
  R w[3][4];
  R pos[3] = {x, y, z};
  // Galerkin ("energy-conserving") variant: order n-1 along every axis on which the component is
  // staggered, order n along the others (it is the gather whose weights equal the
  // Esirkepov deposit's in the limit of a small move, see pin T14)
  int nd[3];
  for (int d = 0; d < 3; ++d) {
    nd[d] = (s.gather_mode == 1 && kStag[comp][d] != 0.0) ? n - 1 : n;
    R xi = pos[d] * s.inv_dx[d] - R(kStag[comp][d]);
    shape<R>(nd[d], xi, &l[d], w[d]);
  }
  R acc = 0;
  for (int c = 0; c <= nd[2]; ++c)
    for (int b = 0; b <= nd[1]; ++b)
      for (int a = 0; a <= nd[0]; ++a)
        acc += w[0][a] * w[1][b] * w[2][c] * s.rd(s.F[comp], l[0] + a, l[1] + b, l[2] + c);
  return acc;
}

// ---------------------------------------------------------------- step 2c
// Relativistic Boris rotation (reading Q2; u = gamma*v in m/s).
template <class R>
void boris(R kq, R inv_c2, const R E[3], const R B[3], R u[3]) {
  R um[3], t[3], up[3], sv[3], upl[3];
  for (int d = 0; d < 3; ++d) um[d] = u[d] + kq * E[d];
  R g = std::sqrt(R(1) + (um[0] * um[0] + um[1] * um[1] + um[2] * um[2]) * inv_c2);
  for (int d = 0; d < 3; ++d) t[d] = kq * B[d] / g;
  up[0] = um[0] + (um[1] * t[2] - um[2] * t[1]);
  up[1] = um[1] + (um[2] * t[0] - um[0] * t[2]);
  up[2] = um[2] + (um[0] * t[1] - um[1] * t[0]);
  R t2 = t[0] * t[0] + t[1] * t[1] + t[2] * t[2];
  for (int d = 0; d < 3; ++d) sv[d] = R(2) * t[d] / (R(1) + t2);
  upl[0] = um[0] + (up[1] * sv[2] - up[2] * sv[1]);
  upl[1] = um[1] + (up[2] * sv[0] - up[0] * sv[2]);
  upl[2] = um[2] + (up[0] * sv[1] - up[1] * sv[0]);
  for (int d = 0; d < 3; ++d) u[d] = upl[d] + kq * E[d];
}

// Vay pusher ("Vay pusher", ref [21] = J.-L. Vay, Phys. Plasmas 15, 056701 (2008));
// u = gamma*v in m/s, kq = q*dt/(2m), in the paper's order:
//   u' = u + 2 kq E + kq (u/gamma) x B;  tau = kq B;  u* = u'.tau / c;  gamma' = sqrt(1 + u'^2/c^2)
//   sigma = gamma'^2 - tau^2;  gamma_new = sqrt((sigma + sqrt(sigma^2 + 4 (tau^2 + u*^2))) / 2)
//   t = tau / gamma_new;  u_new = (u' + (u'.t) t + u' x t) / (1 + t^2)
template <class R>
void vay(R kq, R inv_c2, const R E[3], const R B[3], R u[3]) {
  R g0 = std::sqrt(R(1) + (u[0] * u[0] + u[1] * u[1] + u[2] * u[2]) * inv_c2);
  R v[3] = {u[0] / g0, u[1] / g0, u[2] / g0};
  R up[3], tau[3], t[3];
  up[0] = u[0] + R(2) * kq * E[0] + kq * (v[1] * B[2] - v[2] * B[1]);
  up[1] = u[1] + R(2) * kq * E[1] + kq * (v[2] * B[0] - v[0] * B[2]);
  up[2] = u[2] + R(2) * kq * E[2] + kq * (v[0] * B[1] - v[1] * B[0]);
  for (int d = 0; d < 3; ++d) tau[d] = kq * B[d];
  R tau2 = tau[0] * tau[0] + tau[1] * tau[1] + tau[2] * tau[2];
  R us = (up[0] * tau[0] + up[1] * tau[1] + up[2] * tau[2]) * std::sqrt(inv_c2);
  R gp2 = R(1) + (up[0] * up[0] + up[1] * up[1] + up[2] * up[2]) * inv_c2;
  R sigma = gp2 - tau2;
  R gn = std::sqrt((sigma + std::sqrt(sigma * sigma + R(4) * (tau2 + us * us))) / R(2));
  for (int d = 0; d < 3; ++d) t[d] = tau[d] / gn;
  R t2 = t[0] * t[0] + t[1] * t[1] + t[2] * t[2];
  R ut = up[0] * t[0] + up[1] * t[1] + up[2] * t[2];
  R sc = R(1) / (R(1) + t2);
  u[0] = sc * (up[0] + ut * t[0] + (up[1] * t[2] - up[2] * t[1]));
  u[1] = sc * (up[1] + ut * t[1] + (up[2] * t[0] - up[0] * t[2]));
  u[2] = sc * (up[2] + ut * t[2] + (up[0] * t[1] - up[1] * t[0]));
}

// ---------------------------------------------------------------- step 2e
// Esirkepov charge-conserving deposit of one particle moving x0 -> x1
// (x1 unwrapped), nodal shapes of order n, (n+3)-wide window per axis with
// base b = l0-1 (reading Q5). J accumulates in double (reading Q10).
template <class R, class Sink>
void deposit_to(const Sim<R>& s, const Species<R>& sp, const R x0[3], const R x1[3], R wq, Sink&& add) {
  const int n = s.order, W = n + 3;
  R S0[3][6], S1[3][6], DS[3][6];
  int b[3];
  for (int d = 0; d < 3; ++d) {
    int l0, l1;
    R w0[4], w1[4];
    shape<R>(n, x0[d] * s.inv_dx[d], &l0, w0);
    shape<R>(n, x1[d] * s.inv_dx[d], &l1, w1);
    b[d] = l0 - 1;
    for (int i = 0; i < 6; ++i) { S0[d][i] = 0; S1[d][i] = 0; }
    for (int a = 0; a <= n; ++a) {
      S0[d][1 + a] = w0[a];
      int sl = l1 - b[d] + a;           // in 0..n+2 because |l1-l0|<=1 (CFL)
      if (sl >= 0 && sl < W) S1[d][sl] = w1[a];
    }
    for (int i = 0; i < W; ++i) DS[d][i] = S1[d][i] - S0[d][i];
  }
  const R half = R(0.5), third = R(1) / R(3);
  // Jx: prefix along i
  for (int k = 0; k < W; ++k)
    for (int j = 0; j < W; ++j) {
      R pre = 0;
      for (int i = 0; i < W; ++i) {
        R Wx = DS[0][i] * (S0[1][j] * S0[2][k] + half * DS[1][j] * S0[2][k] +
                           half * S0[1][j] * DS[2][k] + third * DS[1][j] * DS[2][k]);
        pre += Wx;
        add(0, b[0] + i, b[1] + j, b[2] + k, (double)(-(wq * sp.jf[0]) * pre));
      }
    }
  // Jy: prefix along j
  for (int k = 0; k < W; ++k)
    for (int i = 0; i < W; ++i) {
      R pre = 0;
      for (int j = 0; j < W; ++j) {
        R Wy = DS[1][j] * (S0[0][i] * S0[2][k] + half * DS[0][i] * S0[2][k] +
                           half * S0[0][i] * DS[2][k] + third * DS[0][i] * DS[2][k]);
        pre += Wy;
        add(1, b[0] + i, b[1] + j, b[2] + k, (double)(-(wq * sp.jf[1]) * pre));
      }
    }
  // Jz: prefix along k
  for (int j = 0; j < W; ++j)
    for (int i = 0; i < W; ++i) {
      R pre = 0;
      for (int k = 0; k < W; ++k) {
        R Wz = DS[2][k] * (S0[0][i] * S0[1][j] + half * DS[0][i] * S0[1][j] +
                           half * S0[0][i] * DS[1][j] + third * DS[0][i] * DS[1][j]);
        pre += Wz;
        add(2, b[0] + i, b[1] + j, b[2] + k, (double)(-(wq * sp.jf[2]) * pre));
      }
    }
}

// the canonical (serial) sink: straight into the global J, index rule of reading Q6
template <class R>
void deposit(Sim<R>& s, const Species<R>& sp, const R x0[3], const R x1[3], R wq) {
  deposit_to<R>(s, sp, x0, x1, wq, [&](int c, int i, int j, int k, double v) {
    int64_t t = s.lin(i, j, k);
    if (t >= 0) s.Jd[c][(size_t)t] += v;
  });
}

// ---------------------------------------------------------------- S-rules
// Cell of a position: one rounded multiply, floor, clamp (SURVEY.md §8(c) S-rules).
template <class R>
int cell_of(const Sim<R>& s, int d, R x) {
  R p = x * s.inv_dx[d];
  int c = (int)std::floor(p);
  if (c < 0) c = 0;
  if (c > s.N[d] - 1) c = s.N[d] - 1;
  return c;
}

// Stable counting sort by (tile-major) cell key ("counting sort";
// PAPER.md:201 "sort by PIC cell"). perm[k] = old index landing in slot k.
template <class R>
void sort_species(Sim<R>& s, Species<R>& sp) {
  size_t np = sp.x.size();
  const int* T = s.tile;
  int nt[3] = {s.N[0] / T[0], s.N[1] / T[1], s.N[2] / T[2]};
  int64_t tvol = (int64_t)T[0] * T[1] * T[2];
  int64_t nbins = (int64_t)nt[0] * nt[1] * nt[2] * (s.key_mode == 0 ? tvol : 1);
  std::vector<int64_t> key(np);
  sp.cell.assign(np, 0);
  sp.perm.assign(np, 0);
#pragma omp parallel for num_threads(s.omp_threads) if (s.omp_threads > 1) schedule(static)
  for (int64_t p = 0; p < (int64_t)np; ++p) {
    int c[3] = {cell_of(s, 0, sp.x[p]), cell_of(s, 1, sp.y[p]), cell_of(s, 2, sp.z[p])};
    sp.cell[p] = c[0] + s.N[0] * (c[1] + s.N[1] * c[2]);
    int64_t t = (c[0] / T[0]) + (int64_t)nt[0] * ((c[1] / T[1]) + (int64_t)nt[1] * (c[2] / T[2]));
    int64_t r = (c[0] % T[0]) + (int64_t)T[0] * ((c[1] % T[1]) + (int64_t)T[1] * (c[2] % T[2]));
    key[p] = s.key_mode == 0 ? t * tvol + r : t;
  }
  std::vector<int64_t> offs((size_t)nbins + 1, 0);
  for (size_t p = 0; p < np; ++p) offs[(size_t)key[p] + 1]++;            // histogram
  for (int64_t bn = 0; bn < nbins; ++bn) offs[(size_t)bn + 1] += offs[(size_t)bn];  // scan
  for (size_t p = 0; p < np; ++p) sp.perm[(size_t)offs[(size_t)key[p]]++] = (int32_t)p;  // stable scatter
  // gather all arrays and id through perm; `cell` is stored in the new order
  auto permute = [&](auto& v) {
    auto old = v;
#pragma omp parallel for num_threads(s.omp_threads) if (s.omp_threads > 1) schedule(static)
    for (int64_t k = 0; k < (int64_t)np; ++k) v[(size_t)k] = old[(size_t)sp.perm[(size_t)k]];
  };
  permute(sp.x); permute(sp.y); permute(sp.z);
  permute(sp.ux); permute(sp.uy); permute(sp.uz);
  permute(sp.w); permute(sp.id); permute(sp.cell);
}

// ---------------------------------------------------------------- steps 3-5
// Yee curl updates (SURVEY.md §8(c) steps 3,4; forward differences for B,
// backward for E; ref [28] PAPER.md:323).
template <class R>
void push_B_half(Sim<R>& s) {
  auto &Ex = s.F[0], &Ey = s.F[1], &Ez = s.F[2];
  std::vector<R> nBx(s.F[3]), nBy(s.F[4]), nBz(s.F[5]);
#pragma omp parallel for num_threads(s.omp_threads) if (s.omp_threads > 1) schedule(static)
  for (int k = 0; k < s.N[2]; ++k)
    for (int j = 0; j < s.N[1]; ++j)
      for (int i = 0; i < s.N[0]; ++i) {
        size_t t = (size_t)s.lin(i, j, k);
        R ex = Ex[t], ey = Ey[t], ez = Ez[t];
        nBx[t] -= s.cB[1] * (s.rd(Ez, i, j + 1, k) - ez) - s.cB[2] * (s.rd(Ey, i, j, k + 1) - ey);
        nBy[t] -= s.cB[2] * (s.rd(Ex, i, j, k + 1) - ex) - s.cB[0] * (s.rd(Ez, i + 1, j, k) - ez);
        nBz[t] -= s.cB[0] * (s.rd(Ey, i + 1, j, k) - ey) - s.cB[1] * (s.rd(Ex, i, j + 1, k) - ex);
      }
  s.F[3].swap(nBx); s.F[4].swap(nBy); s.F[5].swap(nBz);
}

// CKC solver (PAPER.md:255 lists it among WarpX's solvers; ref [12] Cowan et al., PRST-AB 16, 041303):
// the E update is Yee's; in the B update every difference of E along an axis a is replaced by the
// smoothed difference
//   D_a F = alpha_a dF(0,0) + beta_ab [dF(+b) + dF(-b)] + beta_ac [dF(+c) + dF(-c)]
//         + gamma_a [dF(+b,+c) + dF(+b,-c) + dF(-b,+c) + dF(-b,-c)],   dF(s) = F[+1 along a, s] - F[s],
// b, c the two transverse axes. Coefficients (delta = min dx, r_a = (delta/dx_a)^2, S = r_y r_z + r_z r_x + r_x r_y):
//   beta = (1 - r_x r_y r_z / S) / 8,  beta_ab = r_b beta,  gamma_a = r_b r_c (1/16 - r_b r_c / (8 S)),
//   alpha_a = 1 - 2 beta_ab - 2 beta_ac - 4 gamma_a   (cubic cells: 7/12, 1/12, 1/48).
// They remove the dispersion along the axes at c dt = delta, where the scheme is still stable (pin T15).
template <class R>
R ckc_diff(const Sim<R>& s, const std::vector<R>& F, int a, int i, int j, int k) {
  const int b = (a + 1) % 3, c = (a + 2) % 3;
  auto dF = [&](int sb, int sc) {
    int p[3] = {i, j, k};
    p[b] += sb; p[c] += sc;
    int q[3] = {p[0], p[1], p[2]};
    q[a] += 1;
    return s.rd(F, q[0], q[1], q[2]) - s.rd(F, p[0], p[1], p[2]);
  };
  return s.ck_a[a] * dF(0, 0) + s.ck_b[a][b] * (dF(1, 0) + dF(-1, 0)) + s.ck_b[a][c] * (dF(0, 1) + dF(0, -1)) +
         s.ck_g[a] * (dF(1, 1) + dF(1, -1) + dF(-1, 1) + dF(-1, -1));
}

template <class R>
void push_B_half_ckc(Sim<R>& s) {
  auto &Ex = s.F[0], &Ey = s.F[1], &Ez = s.F[2];
  std::vector<R> nBx(s.F[3]), nBy(s.F[4]), nBz(s.F[5]);
#pragma omp parallel for num_threads(s.omp_threads) if (s.omp_threads > 1) schedule(static)
  for (int k = 0; k < s.N[2]; ++k)
    for (int j = 0; j < s.N[1]; ++j)
      for (int i = 0; i < s.N[0]; ++i) {
        size_t t = (size_t)s.lin(i, j, k);
        nBx[t] -= s.cB[1] * ckc_diff<R>(s, Ez, 1, i, j, k) - s.cB[2] * ckc_diff<R>(s, Ey, 2, i, j, k);
        nBy[t] -= s.cB[2] * ckc_diff<R>(s, Ex, 2, i, j, k) - s.cB[0] * ckc_diff<R>(s, Ez, 0, i, j, k);
        nBz[t] -= s.cB[0] * ckc_diff<R>(s, Ey, 0, i, j, k) - s.cB[1] * ckc_diff<R>(s, Ex, 1, i, j, k);
      }
  s.F[3].swap(nBx); s.F[4].swap(nBy); s.F[5].swap(nBz);
}

template <class R>
void push_B(Sim<R>& s) {
  if (s.solver == 1) push_B_half_ckc<R>(s);
  else push_B_half<R>(s);
}

template <class R>
void push_E(Sim<R>& s) {
  auto &Bx = s.F[3], &By = s.F[4], &Bz = s.F[5];
#pragma omp parallel for num_threads(s.omp_threads) if (s.omp_threads > 1) schedule(static)
  for (int k = 0; k < s.N[2]; ++k)
    for (int j = 0; j < s.N[1]; ++j)
      for (int i = 0; i < s.N[0]; ++i) {
        size_t t = (size_t)s.lin(i, j, k);
        R bx = Bx[t], by = By[t], bz = Bz[t];
        s.F[0][t] += s.cE[1] * (bz - s.rd(Bz, i, j - 1, k)) - s.cE[2] * (by - s.rd(By, i, j, k - 1)) - s.cJ * s.J[0][t];
        s.F[1][t] += s.cE[2] * (bx - s.rd(Bx, i, j, k - 1)) - s.cE[0] * (bz - s.rd(Bz, i - 1, j, k)) - s.cJ * s.J[1][t];
        s.F[2][t] += s.cE[0] * (by - s.rd(By, i - 1, j, k)) - s.cE[1] * (bx - s.rd(Bx, i, j - 1, k)) - s.cJ * s.J[2][t];
      }
}

// ---------------------------------------------------------------- one step
// steps 2b-2g for particle p of one species; `add` receives the particle's J contributions (step 2e)
template <class R, class Sink>
inline void particle_one(const Sim<R>& s, Species<R>& sp, size_t p, Sink&& add, int64_t& n_deactivated) {
  R x0[3] = {sp.x[p], sp.y[p], sp.z[p]};
  R u[3] = {sp.ux[p], sp.uy[p], sp.uz[p]};
  R E[3], B[3];
  for (int c = 0; c < 3; ++c) {                        // 2b
    E[c] = gather<R>(s, c, x0[0], x0[1], x0[2]);
    B[c] = gather<R>(s, 3 + c, x0[0], x0[1], x0[2]);
  }
  if (s.pusher == 1) vay<R>(sp.kq, s.inv_c2, E, B, u);
  else boris<R>(sp.kq, s.inv_c2, E, B, u);             // 2c
  R g = std::sqrt(R(1) + (u[0] * u[0] + u[1] * u[1] + u[2] * u[2]) * s.inv_c2);
  R x1[3];
  for (int d = 0; d < 3; ++d) x1[d] = x0[d] + s.dtr * u[d] / g;   // 2d (unwrapped)
  R w = sp.w[p];
  deposit_to<R>(s, sp, x0, x1, w, add);                // 2e
  for (int d = 0; d < 3; ++d) {                        // 2f
    if (s.periodic[d]) {
      if (x1[d] < R(0)) x1[d] += s.L[d];
      if (x1[d] >= s.L[d]) x1[d] -= s.L[d];
    } else if (!(x1[d] >= R(0) && x1[d] < s.L[d])) {
      if (w != R(0)) n_deactivated++;
      w = R(0);
      x1[d] = x1[d] < R(0) ? R(0) : std::nextafter(s.L[d], R(0));
    }
  }
  sp.x[p] = x1[0]; sp.y[p] = x1[1]; sp.z[p] = x1[2];   // 2g
  sp.ux[p] = u[0]; sp.uy[p] = u[1]; sp.uz[p] = u[2];
  sp.w[p] = w;
}

// the canonical oracle: every particle in current array order, contributions summed straight into J
template <class R>
void particles_step(Sim<R>& s) {
  auto into_J = [&](int c, int i, int j, int k, double v) {
    int64_t t = s.lin(i, j, k);
    if (t >= 0) s.Jd[c][(size_t)t] += v;
  };
  for (auto& sp : s.sp)
    for (size_t p = 0; p < sp.x.size(); ++p) particle_one<R>(s, sp, p, into_J, s.n_deactivated);
}

// ---------------------------------------------------------------- OpenMP variant (pin T12)
// The paper's CPU scheme: the particles are binned onto tiles, OpenMP threads take
// tiles, each thread deposits its tile's particles onto a PRIVATE buffer with enough cells to capture the
// support of every particle of the tile (no atomics), and then adds the buffer to the full grid with one
// atomic per CELL instead of one per particle-node. The per-particle arithmetic is particle_one, unchanged;
// only the order in which contributions reach J differs from the canonical oracle, so the two agree to
// summation roundoff (T12: 1e-13 of max). Used for the N-core baseline of bench.py, never as the checker.
template <class R>
void particles_step_omp(Sim<R>& s, int nthreads) {
  const int* T = s.tile;
  const int nt[3] = {s.N[0] / T[0], s.N[1] / T[1], s.N[2] / T[2]};
  const int64_t ntiles = (int64_t)nt[0] * nt[1] * nt[2];
  // nodes a particle of cell c can touch: c-2 .. c+4 (order 2: l0 in {c-1, c}, window l0-1 .. l0+n+1)
  const int lo = 2, ext[3] = {T[0] + 7, T[1] + 7, T[2] + 7};
  const size_t bvol = (size_t)ext[0] * ext[1] * ext[2];
  for (auto& sp : s.sp) {
    const size_t np = sp.x.size();
    // bin the particles onto tiles by their current cell (stable: ascending index inside a tile)
    std::vector<int64_t> start((size_t)ntiles + 1, 0);
    std::vector<int32_t> tile_of(np), list(np);
#pragma omp parallel for num_threads(nthreads) schedule(static)
    for (int64_t p = 0; p < (int64_t)np; ++p) {
      int c[3] = {cell_of(s, 0, sp.x[p]), cell_of(s, 1, sp.y[p]), cell_of(s, 2, sp.z[p])};
      tile_of[p] = (int32_t)((c[0] / T[0]) + (int64_t)nt[0] * ((c[1] / T[1]) + (int64_t)nt[1] * (c[2] / T[2])));
    }
    for (size_t p = 0; p < np; ++p) start[(size_t)tile_of[p] + 1]++;
    for (int64_t t = 0; t < ntiles; ++t) start[(size_t)t + 1] += start[(size_t)t];
    {
      std::vector<int64_t> fill(start.begin(), start.end() - 1);
      for (size_t p = 0; p < np; ++p) list[(size_t)fill[(size_t)tile_of[p]]++] = (int32_t)p;
    }
    int64_t deact = 0;
#pragma omp parallel num_threads(nthreads) reduction(+ : deact)
    {
      std::vector<double> buf[3];
      for (int c = 0; c < 3; ++c) buf[c].assign(bvol, 0.0);
#pragma omp for schedule(dynamic, 1)
      for (int64_t t = 0; t < ntiles; ++t) {
        if (start[(size_t)t] == start[(size_t)t + 1]) continue;
        const int t0[3] = {(int)(t % nt[0]) * T[0] - lo, (int)((t / nt[0]) % nt[1]) * T[1] - lo,
                           (int)(t / ((int64_t)nt[0] * nt[1])) * T[2] - lo};
        auto into_buf = [&](int c, int i, int j, int k, double v) {
          buf[c][(size_t)(i - t0[0]) + (size_t)ext[0] * ((size_t)(j - t0[1]) + (size_t)ext[1] * (size_t)(k - t0[2]))] += v;
        };
        for (int64_t q = start[(size_t)t]; q < start[(size_t)t + 1]; ++q)
          particle_one<R>(s, sp, (size_t)list[(size_t)q], into_buf, deact);
        // flush: one atomic per touched cell, index rule of reading Q6 (modulo / dropped)
        for (int c = 0; c < 3; ++c)
          for (int k = 0; k < ext[2]; ++k)
            for (int j = 0; j < ext[1]; ++j)
              for (int i = 0; i < ext[0]; ++i) {
                double& v = buf[c][(size_t)i + (size_t)ext[0] * ((size_t)j + (size_t)ext[1] * (size_t)k)];
                if (v == 0.0) continue;
                int64_t g = s.lin(t0[0] + i, t0[1] + j, t0[2] + k);
                if (g >= 0) {
#pragma omp atomic
                  s.Jd[c][(size_t)g] += v;
                }
                v = 0.0;
              }
      }
    }
    s.n_deactivated += deact;
  }
}

// nthreads = 1: the canonical serial oracle. nthreads > 1: the OpenMP variant (particles by tile with private
// J buffers; the node loops of the field solver and the gathers of the sort split over threads — every
// node / slot is independent, so those are bit-identical to the serial loops).
template <class R>
void step(Sim<R>& s, int nthreads = 1) {
  s.omp_threads = nthreads;
  if (s.sort_interval > 0 && s.step_count % s.sort_interval == 0)   // 0
    for (auto& sp : s.sp) sort_species<R>(s, sp);
  for (int c = 0; c < 3; ++c) std::fill(s.Jd[c].begin(), s.Jd[c].end(), 0.0);  // 1
  if (nthreads > 1) particles_step_omp<R>(s, nthreads);
  else particles_step<R>(s);                                        // 2
  for (int c = 0; c < 3; ++c)
    for (size_t t = 0; t < s.ncell(); ++t) s.J[c][t] = (R)s.Jd[c][t];
  push_B<R>(s);                                                     // 3
  push_E<R>(s);                                                     // 4
  push_B<R>(s);                                                     // 5
  s.step_count++;
}

// ---------------------------------------------------------------- diagnostics
// Nodal charge density with the same order-n shape (used by T5/T8 and the
// Gauss residual). Always double.
template <class R>
void deposit_rho(const Sim<R>& s, std::vector<double>& rho) {
  rho.assign(s.ncell(), 0.0);
  double inv_dv = 1.0 / (s.dx[0] * s.dx[1] * s.dx[2]);
  int n = s.order;
  for (auto& sp : s.sp)
    for (size_t p = 0; p < sp.x.size(); ++p) {
      int l[3];
      R w[3][4];
      R pos[3] = {sp.x[p], sp.y[p], sp.z[p]};
      for (int d = 0; d < 3; ++d) shape<R>(n, pos[d] * s.inv_dx[d], &l[d], w[d]);
      for (int c = 0; c <= n; ++c)
        for (int b = 0; b <= n; ++b)
          for (int a = 0; a <= n; ++a) {
            int64_t t = s.lin(l[0] + a, l[1] + b, l[2] + c);
            if (t >= 0) rho[(size_t)t] += sp.q * (double)sp.w[p] * inv_dv * (double)(w[0][a] * w[1][b] * w[2][c]);
          }
    }
}

enum { D_FIELD_E = 0, D_FIELD_B, D_KINETIC, D_CHARGE, D_GAUSS_MAX, D_RHO_MAX, D_DEACT, D_STEPS, D_N };

template <class R>
void diagnostics(const Sim<R>& s, double* out) {
  double dv = s.dx[0] * s.dx[1] * s.dx[2];
  double e2 = 0, b2 = 0;
  for (int c = 0; c < 3; ++c)
    for (size_t t = 0; t < s.ncell(); ++t) {
      e2 += (double)s.F[c][t] * (double)s.F[c][t];
      b2 += (double)s.F[3 + c][t] * (double)s.F[3 + c][t];
    }
  out[D_FIELD_E] = 0.5 * kEps0 * e2 * dv;
  out[D_FIELD_B] = 0.5 * kEps0 * kC * kC * b2 * dv;
  double ke = 0, ch = 0;
  for (auto& sp : s.sp)
    for (size_t p = 0; p < sp.x.size(); ++p) {
      double u2 = (double)sp.ux[p] * sp.ux[p] + (double)sp.uy[p] * sp.uy[p] + (double)sp.uz[p] * sp.uz[p];
      double a = u2 / (kC * kC);
      double gm1 = a / (1.0 + std::sqrt(1.0 + a));     // gamma-1 without cancellation
      ke += (double)sp.w[p] * sp.m * kC * kC * gm1;
      ch += sp.q * (double)sp.w[p];
    }
  out[D_KINETIC] = ke;
  out[D_CHARGE] = ch;
  std::vector<double> rho;
  deposit_rho<R>(s, rho);
  double gmax = 0, rmax = 0;
  for (int k = 0; k < s.N[2]; ++k)
    for (int j = 0; j < s.N[1]; ++j)
      for (int i = 0; i < s.N[0]; ++i) {
        size_t t = (size_t)s.lin(i, j, k);
        double div = ((double)s.F[0][t] - (double)s.rd(s.F[0], i - 1, j, k)) / s.dx[0] +
                     ((double)s.F[1][t] - (double)s.rd(s.F[1], i, j - 1, k)) / s.dx[1] +
                     ((double)s.F[2][t] - (double)s.rd(s.F[2], i, j, k - 1)) / s.dx[2];
        gmax = std::max(gmax, std::fabs(div - rho[t] / kEps0));
        rmax = std::max(rmax, std::fabs(rho[t] / kEps0));
      }
  out[D_GAUSS_MAX] = gmax;
  out[D_RHO_MAX] = rmax;
  out[D_DEACT] = (double)s.n_deactivated;
  out[D_STEPS] = (double)s.step_count;
}

// ---------------------------------------------------------------- handle
struct Handle {
  int prec;            // 0 = f64, 1 = f32
  Sim<double>* d = nullptr;
  Sim<float>* f = nullptr;
  std::string err;
};

template <class R>
Sim<R>* make_sim(const int32_t* N, const double* dx, double dt, int order, const int32_t* periodic,
                 const int32_t* tile, int sort_interval, int key_mode) {
  auto* s = new Sim<R>();
  for (int d = 0; d < 3; ++d) {
    s->N[d] = N[d]; s->dx[d] = dx[d];
    s->periodic[d] = periodic[d]; s->tile[d] = tile[d];
    s->inv_dx[d] = (R)(1.0 / dx[d]);
    s->L[d] = (R)(N[d] * dx[d]);
    s->cB[d] = (R)(dt / (2.0 * dx[d]));
    s->cE[d] = (R)(kC * kC * dt / dx[d]);
  }
  {
    const double delta = std::min(dx[0], std::min(dx[1], dx[2]));
    double r[3];
    for (int d = 0; d < 3; ++d) r[d] = (delta / dx[d]) * (delta / dx[d]);
    const double S = r[1] * r[2] + r[2] * r[0] + r[0] * r[1];
    const double beta = 0.125 * (1.0 - r[0] * r[1] * r[2] / S);
    for (int a = 0; a < 3; ++a) {
      const int b = (a + 1) % 3, c = (a + 2) % 3;
      const double bab = r[b] * beta, bac = r[c] * beta;
      const double ga = r[b] * r[c] * (0.0625 - 0.125 * r[b] * r[c] / S);
      s->ck_b[a][a] = R(0); s->ck_b[a][b] = (R)bab; s->ck_b[a][c] = (R)bac;
      s->ck_g[a] = (R)ga;
      s->ck_a[a] = (R)(1.0 - 2.0 * bab - 2.0 * bac - 4.0 * ga);
    }
  }
  s->dt = dt; s->order = order; s->sort_interval = sort_interval; s->key_mode = key_mode;
  s->cJ = (R)(dt / kEps0);
  s->inv_c2 = (R)(1.0 / (kC * kC));
  s->dtr = (R)dt;
  for (int c = 0; c < 6; ++c) s->F[c].assign(s->ncell(), R(0));
  for (int c = 0; c < 3; ++c) { s->Jd[c].assign(s->ncell(), 0.0); s->J[c].assign(s->ncell(), R(0)); }
  return s;
}

template <class R>
int add_species(Sim<R>& s, int64_t n, const void* const* arr, double q, double m) {
  Species<R> sp;
  sp.q = q; sp.m = m;
  sp.kq = (R)(q * s.dt / (2.0 * m));
  sp.jf[0] = (R)(q / (s.dt * s.dx[1] * s.dx[2]));
  sp.jf[1] = (R)(q / (s.dt * s.dx[0] * s.dx[2]));
  sp.jf[2] = (R)(q / (s.dt * s.dx[0] * s.dx[1]));
  std::vector<R>* dst[7] = {&sp.x, &sp.y, &sp.z, &sp.ux, &sp.uy, &sp.uz, &sp.w};
  for (int a = 0; a < 7; ++a) {
    const R* src = (const R*)arr[a];
    dst[a]->assign(src, src + n);
  }
  sp.id.resize((size_t)n);
  for (int64_t p = 0; p < n; ++p) sp.id[(size_t)p] = p;
  s.sp.push_back(std::move(sp));
  return (int)s.sp.size() - 1;
}

}  // namespace

#define DISPATCH(h, expr_d, expr_f) ((h)->prec == 0 ? (expr_d) : (expr_f))

extern "C" {

// --- whole-simulation interface (mirrors the product's calls; reading SURVEY.md §8(b))
// solver: 0 Yee (stable for c dt sqrt(sum 1/dx^2) <= 1), 1 CKC (stable for c dt <= min dx)
void* orc_create_ex(const int32_t* n_cells, const double* dx, double dt, int order, int prec,
                    const int32_t* periodic, const int32_t* tile, int sort_interval, int key_mode, int solver) {
  if (order < 1 || order > 3) return nullptr;
  for (int d = 0; d < 3; ++d)
    if (n_cells[d] < 1 || tile[d] < 1 || n_cells[d] % tile[d] != 0 || !(dx[d] > 0)) return nullptr;
  double s2 = 0;
  for (int d = 0; d < 3; ++d) s2 += 1.0 / (dx[d] * dx[d]);
  if (solver < 0 || solver > 1) return nullptr;
  const double dmin = std::min(dx[0], std::min(dx[1], dx[2]));
  if (!(dt > 0) || (solver == 0 ? dt * kC * std::sqrt(s2) > 1.0 : dt * kC > dmin * (1.0 + 1e-12))) return nullptr;   // CFL
  auto* h = new Handle();
  h->prec = prec;
  if (prec == 0) h->d = make_sim<double>(n_cells, dx, dt, order, periodic, tile, sort_interval, key_mode);
  else h->f = make_sim<float>(n_cells, dx, dt, order, periodic, tile, sort_interval, key_mode);
  if (prec == 0) h->d->solver = solver; else h->f->solver = solver;
  return h;
}

void* orc_create(const int32_t* n_cells, const double* dx, double dt, int order, int prec,
                 const int32_t* periodic, const int32_t* tile, int sort_interval, int key_mode) {
  return orc_create_ex(n_cells, dx, dt, order, prec, periodic, tile, sort_interval, key_mode, 0);
}

// CKC coefficients as the oracle uses them (f64): out[0..2] alpha_a, out[3..11] beta_ab row-major, out[12..14] gamma_a
void orc_ckc_coefficients(void* hv, double* out) {
  auto* h = (Handle*)hv;
  for (int a = 0; a < 3; ++a) {
    out[a] = h->prec == 0 ? (double)h->d->ck_a[a] : (double)h->f->ck_a[a];
    out[12 + a] = h->prec == 0 ? (double)h->d->ck_g[a] : (double)h->f->ck_g[a];
    for (int b = 0; b < 3; ++b) out[3 + 3 * a + b] = h->prec == 0 ? (double)h->d->ck_b[a][b] : (double)h->f->ck_b[a][b];
  }
}

void orc_destroy(void* hv) {
  auto* h = (Handle*)hv;
  if (!h) return;
  delete h->d; delete h->f; delete h;
}

int orc_add_species(void* hv, int64_t n, const void* x, const void* y, const void* z, const void* ux,
                    const void* uy, const void* uz, const void* w, double q, double m) {
  auto* h = (Handle*)hv;
  const void* arr[7] = {x, y, z, ux, uy, uz, w};
  return DISPATCH(h, add_species<double>(*h->d, n, arr, q, m), add_species<float>(*h->f, n, arr, q, m));
}

void orc_set_fields(void* hv, const void* const* E, const void* const* B) {
  auto* h = (Handle*)hv;
  for (int c = 0; c < 3; ++c) {
    if (h->prec == 0) {
      std::memcpy(h->d->F[c].data(), E[c], h->d->ncell() * 8);
      std::memcpy(h->d->F[3 + c].data(), B[c], h->d->ncell() * 8);
    } else {
      std::memcpy(h->f->F[c].data(), E[c], h->f->ncell() * 4);
      std::memcpy(h->f->F[3 + c].data(), B[c], h->f->ncell() * 4);
    }
  }
}

void orc_step(void* hv, int n) {
  auto* h = (Handle*)hv;
  for (int i = 0; i < n; ++i) {
    if (h->prec == 0) step<double>(*h->d); else step<float>(*h->f);
  }
}

// OpenMP variant of orc_step (pin T12); nthreads <= 0: all the threads OpenMP offers.
// Returns the thread count used.
int orc_step_omp(void* hv, int n, int nthreads) {
  auto* h = (Handle*)hv;
  if (nthreads <= 0) nthreads = omp_get_max_threads();
  for (int i = 0; i < n; ++i) {
    if (h->prec == 0) step<double>(*h->d, nthreads); else step<float>(*h->f, nthreads);
  }
  if (h->prec == 0) h->d->omp_threads = 1; else h->f->omp_threads = 1;
  return nthreads;
}

void orc_get_fields(void* hv, void* const* E, void* const* B, void* const* J) {
  auto* h = (Handle*)hv;
  for (int c = 0; c < 3; ++c) {
    if (h->prec == 0) {
      size_t nb = h->d->ncell() * 8;
      if (E) std::memcpy(E[c], h->d->F[c].data(), nb);
      if (B) std::memcpy(B[c], h->d->F[3 + c].data(), nb);
      if (J) std::memcpy(J[c], h->d->J[c].data(), nb);
    } else {
      size_t nb = h->f->ncell() * 4;
      if (E) std::memcpy(E[c], h->f->F[c].data(), nb);
      if (B) std::memcpy(B[c], h->f->F[3 + c].data(), nb);
      if (J) std::memcpy(J[c], h->f->J[c].data(), nb);
    }
  }
}

int64_t orc_num_particles(void* hv, int sp) {
  auto* h = (Handle*)hv;
  return DISPATCH(h, (int64_t)h->d->sp[sp].x.size(), (int64_t)h->f->sp[sp].x.size());
}

void orc_get_particles(void* hv, int isp, void* x, void* y, void* z, void* ux, void* uy, void* uz,
                       void* w, int64_t* id) {
  auto* h = (Handle*)hv;
  void* out[7] = {x, y, z, ux, uy, uz, w};
  if (h->prec == 0) {
    auto& sp = h->d->sp[isp];
    std::vector<double>* src[7] = {&sp.x, &sp.y, &sp.z, &sp.ux, &sp.uy, &sp.uz, &sp.w};
    for (int a = 0; a < 7; ++a) if (out[a]) std::memcpy(out[a], src[a]->data(), src[a]->size() * 8);
    if (id) std::memcpy(id, sp.id.data(), sp.id.size() * 8);
  } else {
    auto& sp = h->f->sp[isp];
    std::vector<float>* src[7] = {&sp.x, &sp.y, &sp.z, &sp.ux, &sp.uy, &sp.uz, &sp.w};
    for (int a = 0; a < 7; ++a) if (out[a]) std::memcpy(out[a], src[a]->data(), src[a]->size() * 4);
    if (id) std::memcpy(id, sp.id.data(), sp.id.size() * 8);
  }
}

// state of the most recent sort: cell[] (linear cell of slot k) and perm[] (old index of slot k)
int orc_get_sort_state(void* hv, int isp, int32_t* cell, int32_t* perm) {
  auto* h = (Handle*)hv;
  const std::vector<int32_t>* c = DISPATCH(h, &h->d->sp[isp].cell, &h->f->sp[isp].cell);
  const std::vector<int32_t>* p = DISPATCH(h, &h->d->sp[isp].perm, &h->f->sp[isp].perm);
  if (c->empty() && orc_num_particles(hv, isp) > 0) return -1;
  if (cell) std::memcpy(cell, c->data(), c->size() * 4);
  if (perm) std::memcpy(perm, p->data(), p->size() * 4);
  return 0;
}

int orc_ndiag() { return D_N; }
void orc_get_diagnostics(void* hv, double* out) {
  auto* h = (Handle*)hv;
  if (h->prec == 0) diagnostics<double>(*h->d, out); else diagnostics<float>(*h->f, out);
}

void orc_get_rho(void* hv, double* rho) {
  auto* h = (Handle*)hv;
  std::vector<double> r;
  if (h->prec == 0) deposit_rho<double>(*h->d, r); else deposit_rho<float>(*h->f, r);
  std::memcpy(rho, r.data(), r.size() * 8);
}

// --- single pieces, exposed so that each can be pinned on its own
// force a sort now (step 0 of the loop, regardless of cadence)
void orc_sort_now(void* hv) {
  auto* h = (Handle*)hv;
  if (h->prec == 0) for (auto& sp : h->d->sp) sort_species<double>(*h->d, sp);
  else for (auto& sp : h->f->sp) sort_species<float>(*h->f, sp);
}
// field solver only (steps 3-5 with J = current J array contents)
void orc_field_step(void* hv, int n) {
  auto* h = (Handle*)hv;
  for (int i = 0; i < n; ++i) {
    if (h->prec == 0) { push_B(*h->d); push_E(*h->d); push_B(*h->d); }
    else { push_B(*h->f); push_E(*h->f); push_B(*h->f); }
  }
}
// zero J, run step 2 for every particle, round J; no sort, no field update
void orc_particle_step(void* hv) {
  auto* h = (Handle*)hv;
  if (h->prec == 0) {
    auto& s = *h->d;
    for (int c = 0; c < 3; ++c) std::fill(s.Jd[c].begin(), s.Jd[c].end(), 0.0);
    particles_step<double>(s);
    for (int c = 0; c < 3; ++c) for (size_t t = 0; t < s.ncell(); ++t) s.J[c][t] = s.Jd[c][t];
  } else {
    auto& s = *h->f;
    for (int c = 0; c < 3; ++c) std::fill(s.Jd[c].begin(), s.Jd[c].end(), 0.0);
    particles_step<float>(s);
    for (int c = 0; c < 3; ++c) for (size_t t = 0; t < s.ncell(); ++t) s.J[c][t] = (float)s.Jd[c][t];
  }
}

void orc_shape_f64(int order, double xi, int32_t* l, double* w) { int ll; shape<double>(order, xi, &ll, w); *l = ll; }
void orc_shape_f32(int order, float xi, int32_t* l, float* w) { int ll; shape<float>(order, xi, &ll, w); *l = ll; }
// pusher: 0 Boris, 1 Vay; gather_mode: 0 uniform order, 1 Galerkin. Returns 0, or -1 for bad values.
int orc_set_method(void* hv, int pusher, int gather_mode) {
  auto* h = (Handle*)hv;
  if (!h || pusher < 0 || pusher > 1 || gather_mode < 0 || gather_mode > 1) return -1;
  if (h->prec == 0) { h->d->pusher = pusher; h->d->gather_mode = gather_mode; }
  else { h->f->pusher = pusher; h->f->gather_mode = gather_mode; }
  return 0;
}
void orc_vay_f64(double kq, const double* E, const double* B, double* u) {
  vay<double>(kq, 1.0 / (kC * kC), E, B, u);
}
void orc_vay_f32(float kq, const float* E, const float* B, float* u) {
  vay<float>(kq, (float)(1.0 / (kC * kC)), E, B, u);
}
void orc_boris_f64(double kq, const double* E, const double* B, double* u) {
  boris<double>(kq, 1.0 / (kC * kC), E, B, u);
}
void orc_boris_f32(float kq, const float* E, const float* B, float* u) {
  boris<float>(kq, (float)(1.0 / (kC * kC)), E, B, u);
}
// gather the six components at arbitrary positions with the sim's current fields
void orc_gather(void* hv, int64_t n, const void* x, const void* y, const void* z, void* out6n) {
  auto* h = (Handle*)hv;
  for (int64_t p = 0; p < n; ++p)
    for (int c = 0; c < 6; ++c) {
      if (h->prec == 0)
        ((double*)out6n)[6 * p + c] = gather<double>(*h->d, c, ((const double*)x)[p], ((const double*)y)[p], ((const double*)z)[p]);
      else
        ((float*)out6n)[6 * p + c] = gather<float>(*h->f, c, ((const float*)x)[p], ((const float*)y)[p], ((const float*)z)[p]);
    }
}
// deposit explicit moves x0->x1 (x1 unwrapped) of species isp's charge with weights w into a
// zeroed J; used by T5-T7
void orc_deposit_moves(void* hv, int isp, int64_t n, const void* x0, const void* x1, const void* w) {
  auto* h = (Handle*)hv;
  if (h->prec == 0) {
    auto& s = *h->d;
    for (int c = 0; c < 3; ++c) std::fill(s.Jd[c].begin(), s.Jd[c].end(), 0.0);
    for (int64_t p = 0; p < n; ++p)
      deposit<double>(s, s.sp[isp], (const double*)x0 + 3 * p, (const double*)x1 + 3 * p, ((const double*)w)[p]);
    for (int c = 0; c < 3; ++c) for (size_t t = 0; t < s.ncell(); ++t) s.J[c][t] = s.Jd[c][t];
  } else {
    auto& s = *h->f;
    for (int c = 0; c < 3; ++c) std::fill(s.Jd[c].begin(), s.Jd[c].end(), 0.0);
    for (int64_t p = 0; p < n; ++p)
      deposit<float>(s, s.sp[isp], (const float*)x0 + 3 * p, (const float*)x1 + 3 * p, ((const float*)w)[p]);
    for (int c = 0; c < 3; ++c) for (size_t t = 0; t < s.ncell(); ++t) s.J[c][t] = (float)s.Jd[c][t];
  }
}
double orc_const_c() { return kC; }
double orc_const_eps0() { return kEps0; }

}  // extern "C"
