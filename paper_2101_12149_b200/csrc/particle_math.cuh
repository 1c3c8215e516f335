// Per-particle device math of the CUDA path: gather, Boris, Esirkepov set-up, wrap
// (steps 2a-2f). Included by particles.cu only.
#pragma once
#include "common.cuh"

namespace pic {

// ------------------------------------------------------------------ gather
// Tensor-product interpolation of one component, nested so each inner sum is reused:
// (n+1)^3 + (n+1)^2 + (n+1) FMAs.
template <class R, int ORDER>
__device__ __forceinline__ R interp(const R* __restrict__ F, int base, int sy, int sz,
                                    const R* wx, const R* wy, const R* wz) {
  R acc = 0;
  if constexpr (kStatementOrder<R>) {   // sum over c, b, a (a innermost) of ((wx wy) wz) F, every operation rounded
#pragma unroll
    for (int c = 0; c <= ORDER; ++c)
#pragma unroll
      for (int b = 0; b <= ORDER; ++b)
#pragma unroll
        for (int a = 0; a <= ORDER; ++a)
          acc = add_rn(acc, mul_rn(mul_rn(mul_rn(wx[a], wy[b]), wz[c]), __ldg(F + base + a + sy * b + sz * c)));
  } else {
#pragma unroll
    for (int c = 0; c <= ORDER; ++c) {
      R accb = 0;
#pragma unroll
      for (int b = 0; b <= ORDER; ++b) {
        R acca = 0;
#pragma unroll
        for (int a = 0; a <= ORDER; ++a) acca += wx[a] * __ldg(F + base + a + sy * b + sz * c);
        accb += wy[b] * acca;
      }
      acc += wz[c] * accb;
    }
  }
  return acc;
}

template <class R, int ORDER, bool GENERIC = true>
__device__ __forceinline__ void gather6(const Grid<R>& g, R x, R y, R z, R* E, R* B) {
  // nodal (offset 0) and staggered (offset 1/2) weight sets per axis, shared by the components
  R wn[3][ORDER + 1], ws[3][ORDER + 1];
  int ln[3], ls[3];
  R pos[3] = {x, y, z};
#pragma unroll
  for (int d = 0; d < 3; ++d) {
    const R xi = mul_rn(pos[d], g.inv_dx[d]);
    const R xs = sub_rn(xi, R(0.5));
    ln[d] = shape<R, ORDER>(xi, wn[d]);
    ls[d] = (GENERIC && g.gather_mode) ? shape_lowered<R, ORDER>(xs, ws[d]) : shape<R, ORDER>(xs, ws[d]);
    // memory safety if a position ever went non-finite: keep the stencil inside the padded box
    ln[d] = min(max(ln[d], -kGuard), g.N[d] + kGuard - ORDER - 1);
    ls[d] = min(max(ls[d], -kGuard), g.N[d] + kGuard - ORDER - 1);
  }
  const int sy = g.sy, sz = g.sz;
  // Ex (s,n,n)  Ey (n,s,n)  Ez (n,n,s)  Bx (n,s,s)  By (s,n,s)  Bz (s,s,n)
  E[0] = interp<R, ORDER>(g.F[0], g.idx(ls[0], ln[1], ln[2]), sy, sz, ws[0], wn[1], wn[2]);
  E[1] = interp<R, ORDER>(g.F[1], g.idx(ln[0], ls[1], ln[2]), sy, sz, wn[0], ws[1], wn[2]);
  E[2] = interp<R, ORDER>(g.F[2], g.idx(ln[0], ln[1], ls[2]), sy, sz, wn[0], wn[1], ws[2]);
  B[0] = interp<R, ORDER>(g.F[3], g.idx(ln[0], ls[1], ls[2]), sy, sz, wn[0], ws[1], ws[2]);
  B[1] = interp<R, ORDER>(g.F[4], g.idx(ls[0], ln[1], ls[2]), sy, sz, ws[0], wn[1], ws[2]);
  B[2] = interp<R, ORDER>(g.F[5], g.idx(ls[0], ls[1], ln[2]), sy, sz, ws[0], ws[1], wn[2]);
}

// ------------------------------------------------------------------ Boris
template <class R>
__device__ __forceinline__ void boris(R kq, R inv_c2, const R* E, const R* B, R* u) {
  if constexpr (kStatementOrder<R>) {
    R um[3], t[3], up[3], sv[3];
#pragma unroll
    for (int d = 0; d < 3; ++d) um[d] = add_rn(u[d], mul_rn(kq, E[d]));
    const R g = sqrt_rn(add_rn(R(1), mul_rn(add_rn(add_rn(mul_rn(um[0], um[0]), mul_rn(um[1], um[1])), mul_rn(um[2], um[2])), inv_c2)));
#pragma unroll
    for (int d = 0; d < 3; ++d) t[d] = div_rn(mul_rn(kq, B[d]), g);
    up[0] = add_rn(um[0], sub_rn(mul_rn(um[1], t[2]), mul_rn(um[2], t[1])));
    up[1] = add_rn(um[1], sub_rn(mul_rn(um[2], t[0]), mul_rn(um[0], t[2])));
    up[2] = add_rn(um[2], sub_rn(mul_rn(um[0], t[1]), mul_rn(um[1], t[0])));
    const R den = add_rn(R(1), add_rn(add_rn(mul_rn(t[0], t[0]), mul_rn(t[1], t[1])), mul_rn(t[2], t[2])));
#pragma unroll
    for (int d = 0; d < 3; ++d) sv[d] = div_rn(mul_rn(R(2), t[d]), den);
    const R v0 = add_rn(um[0], sub_rn(mul_rn(up[1], sv[2]), mul_rn(up[2], sv[1])));
    const R v1 = add_rn(um[1], sub_rn(mul_rn(up[2], sv[0]), mul_rn(up[0], sv[2])));
    const R v2 = add_rn(um[2], sub_rn(mul_rn(up[0], sv[1]), mul_rn(up[1], sv[0])));
    u[0] = add_rn(v0, mul_rn(kq, E[0]));
    u[1] = add_rn(v1, mul_rn(kq, E[1]));
    u[2] = add_rn(v2, mul_rn(kq, E[2]));
    return;
  }
  R um0 = u[0] + kq * E[0], um1 = u[1] + kq * E[1], um2 = u[2] + kq * E[2];
  R ig = R(1) / sqrt(R(1) + (um0 * um0 + um1 * um1 + um2 * um2) * inv_c2);
  R t0 = kq * B[0] * ig, t1 = kq * B[1] * ig, t2 = kq * B[2] * ig;
  R up0 = um0 + (um1 * t2 - um2 * t1);
  R up1 = um1 + (um2 * t0 - um0 * t2);
  R up2 = um2 + (um0 * t1 - um1 * t0);
  R sc = R(2) / (R(1) + (t0 * t0 + t1 * t1 + t2 * t2));
  R s0 = t0 * sc, s1 = t1 * sc, s2 = t2 * sc;
  u[0] = um0 + (up1 * s2 - up2 * s1) + kq * E[0];
  u[1] = um1 + (up2 * s0 - up0 * s2) + kq * E[1];
  u[2] = um2 + (up0 * s1 - up1 * s0) + kq * E[2];
}

// ------------------------------------------------------------------ Vay (ref [21])
// u' = u + 2 kq E + kq (u/gamma) x B; tau = kq B; u* = u'.tau/c; sigma = gamma'^2 - tau^2;
// gamma_new = sqrt((sigma + sqrt(sigma^2 + 4 (tau^2 + u*^2))) / 2); t = tau/gamma_new;
// u_new = (u' + (u'.t) t + u' x t) / (1 + t^2)
template <class R>
__device__ __forceinline__ void vay(R kq, R inv_c2, const R* E, const R* B, R* u) {
  if constexpr (kStatementOrder<R>) {
    auto dot3 = [](const R* a, const R* b) {
      return add_rn(add_rn(mul_rn(a[0], b[0]), mul_rn(a[1], b[1])), mul_rn(a[2], b[2]));
    };
    const R g0 = sqrt_rn(add_rn(R(1), mul_rn(dot3(u, u), inv_c2)));
    const R v[3] = {div_rn(u[0], g0), div_rn(u[1], g0), div_rn(u[2], g0)};
    R up[3], tau[3], t[3];
#pragma unroll
    for (int d = 0; d < 3; ++d) {
      const int a = (d + 1) % 3, b = (d + 2) % 3;
      up[d] = add_rn(add_rn(u[d], mul_rn(mul_rn(R(2), kq), E[d])),
                     mul_rn(kq, sub_rn(mul_rn(v[a], B[b]), mul_rn(v[b], B[a]))));
      tau[d] = mul_rn(kq, B[d]);
    }
    const R tau2 = dot3(tau, tau);
    const R us = mul_rn(dot3(up, tau), sqrt_rn(inv_c2));
    const R gp2 = add_rn(R(1), mul_rn(dot3(up, up), inv_c2));
    const R sigma = sub_rn(gp2, tau2);
    const R gn = sqrt_rn(div_rn(
        add_rn(sigma, sqrt_rn(add_rn(mul_rn(sigma, sigma), mul_rn(R(4), add_rn(tau2, mul_rn(us, us)))))), R(2)));
#pragma unroll
    for (int d = 0; d < 3; ++d) t[d] = div_rn(tau[d], gn);
    const R t2 = dot3(t, t);
    const R ut = dot3(up, t);
    const R sc = div_rn(R(1), add_rn(R(1), t2));
    R un[3];
#pragma unroll
    for (int d = 0; d < 3; ++d) {
      const int a = (d + 1) % 3, b = (d + 2) % 3;
      un[d] = mul_rn(sc, add_rn(add_rn(up[d], mul_rn(ut, t[d])), sub_rn(mul_rn(up[a], t[b]), mul_rn(up[b], t[a]))));
    }
    u[0] = un[0]; u[1] = un[1]; u[2] = un[2];
    return;
  }
  const R ig0 = R(1) / sqrt(R(1) + (u[0] * u[0] + u[1] * u[1] + u[2] * u[2]) * inv_c2);
  const R v0 = u[0] * ig0, v1 = u[1] * ig0, v2 = u[2] * ig0;
  const R up0 = u[0] + R(2) * kq * E[0] + kq * (v1 * B[2] - v2 * B[1]);
  const R up1 = u[1] + R(2) * kq * E[1] + kq * (v2 * B[0] - v0 * B[2]);
  const R up2 = u[2] + R(2) * kq * E[2] + kq * (v0 * B[1] - v1 * B[0]);
  const R ta0 = kq * B[0], ta1 = kq * B[1], ta2 = kq * B[2];
  const R tau2 = ta0 * ta0 + ta1 * ta1 + ta2 * ta2;
  const R us = (up0 * ta0 + up1 * ta1 + up2 * ta2) * sqrt(inv_c2);
  const R gp2 = R(1) + (up0 * up0 + up1 * up1 + up2 * up2) * inv_c2;
  const R sigma = gp2 - tau2;
  const R ign = R(1) / sqrt((sigma + sqrt(sigma * sigma + R(4) * (tau2 + us * us))) * R(0.5));
  const R t0 = ta0 * ign, t1 = ta1 * ign, t2 = ta2 * ign;
  const R ut = up0 * t0 + up1 * t1 + up2 * t2;
  const R sc = R(1) / (R(1) + (t0 * t0 + t1 * t1 + t2 * t2));
  u[0] = sc * (up0 + ut * t0 + (up1 * t2 - up2 * t1));
  u[1] = sc * (up1 + ut * t1 + (up2 * t0 - up0 * t2));
  u[2] = sc * (up2 + ut * t2 + (up0 * t1 - up1 * t0));
}

// step 2c with the pusher the simulation was created with (warp-uniform branch)
template <class R>
__device__ __forceinline__ void push_momentum(int pusher, R kq, R inv_c2, const R* E, const R* B, R* u) {
  if (pusher) vay<R>(kq, inv_c2, E, B, u);
  else boris<R>(kq, inv_c2, E, B, u);
}

// step 2d: x~ = x + dt u / gamma(u), unwrapped
template <class R>
__device__ __forceinline__ void advance(R dt, R inv_c2, const R* x0, const R* u, R* x1) {
  if constexpr (kStatementOrder<R>) {
    const R g = sqrt_rn(add_rn(R(1), mul_rn(add_rn(add_rn(mul_rn(u[0], u[0]), mul_rn(u[1], u[1])), mul_rn(u[2], u[2])), inv_c2)));
#pragma unroll
    for (int d = 0; d < 3; ++d) x1[d] = add_rn(x0[d], div_rn(mul_rn(dt, u[d]), g));
  } else {
    const R ig = dt / sqrt(R(1) + (u[0] * u[0] + u[1] * u[1] + u[2] * u[2]) * inv_c2);
#pragma unroll
    for (int d = 0; d < 3; ++d) x1[d] = x0[d] + u[d] * ig;
  }
}

// ------------------------------------------------------------------ Esirkepov, per axis set-up
// Old and new nodal weights on a COMPACT window of ORDER+2 nodes that starts at grid index
// `base` = min(l0, l1): the (ORDER+3)-wide window of the definition minus the slot that holds
// neither (identical sums; reading Q5).
template <class R, int ORDER>
__device__ __forceinline__ int esirkepov_axis(R xi0, R xi1, R* S0, R* DS) {
  constexpr int NW = ORDER + 2;
  R w0[ORDER + 1], w1[ORDER + 1];
  int l0 = shape<R, ORDER>(xi0, w0);
  int l1 = shape<R, ORDER>(xi1, w1);
  int sh = l1 - l0;                 // -1, 0, +1 (CFL)
  bool o0 = sh < 0;                 // old weights start at slot 1 when the particle moved down
  bool o1 = sh > 0;                 // new weights start at slot 1 when it moved up
#pragma unroll
  for (int i = 0; i < NW; ++i) {
    R a_lo = i <= ORDER ? w0[i <= ORDER ? i : 0] : R(0);
    R a_hi = i >= 1 ? w0[i >= 1 ? i - 1 : 0] : R(0);
    R b_lo = i <= ORDER ? w1[i <= ORDER ? i : 0] : R(0);
    R b_hi = i >= 1 ? w1[i >= 1 ? i - 1 : 0] : R(0);
    S0[i] = o0 ? a_hi : a_lo;
    DS[i] = sub_rn(o1 ? b_hi : b_lo, S0[i]);
  }
  return o0 ? l1 : l0;
}

// One thread per particle, one global reduction per particle-node.
template <class R, int ORDER>
__device__ __forceinline__ void deposit_global(const Grid<R>& g, const R* jf, R wq, const R* x0, const R* x1) {
  constexpr int NW = ORDER + 2;
  R S0[3][NW], DS[3][NW];
  int b[3];
#pragma unroll
  for (int d = 0; d < 3; ++d) {
    b[d] = esirkepov_axis<R, ORDER>(mul_rn(x0[d], g.inv_dx[d]), mul_rn(x1[d], g.inv_dx[d]), S0[d], DS[d]);
    b[d] = min(max(b[d], -kGuard), g.N[d] + kGuard - NW);
  }
  const int base = g.idx(b[0], b[1], b[2]);
  const int sy = g.sy, sz = g.sz;
  const R half = R(0.5), third = R(1) / R(3);
  const R fx = -(wq * jf[0]), fy = -(wq * jf[1]), fz = -(wq * jf[2]);
  R* __restrict__ Jx = g.J[0];
  R* __restrict__ Jy = g.J[1];
  R* __restrict__ Jz = g.J[2];
#pragma unroll
  for (int k = 0; k < NW; ++k)
#pragma unroll
    for (int j = 0; j < NW; ++j) {
      R c = S0[1][j] * S0[2][k] + half * DS[1][j] * S0[2][k] + half * S0[1][j] * DS[2][k] + third * DS[1][j] * DS[2][k];
      R pre = 0;
#pragma unroll
      for (int i = 0; i < NW - 1; ++i) {
        pre += DS[0][i] * c;
        R v = fx * pre;
        if (v != R(0)) j_add<R>(g, Jx + base + i + sy * j + sz * k, v);
      }
    }
#pragma unroll
  for (int k = 0; k < NW; ++k)
#pragma unroll
    for (int i = 0; i < NW; ++i) {
      R c = S0[0][i] * S0[2][k] + half * DS[0][i] * S0[2][k] + half * S0[0][i] * DS[2][k] + third * DS[0][i] * DS[2][k];
      R pre = 0;
#pragma unroll
      for (int j = 0; j < NW - 1; ++j) {
        pre += DS[1][j] * c;
        R v = fy * pre;
        if (v != R(0)) j_add<R>(g, Jy + base + i + sy * j + sz * k, v);
      }
    }
#pragma unroll
  for (int j = 0; j < NW; ++j)
#pragma unroll
    for (int i = 0; i < NW; ++i) {
      R c = S0[0][i] * S0[1][j] + half * DS[0][i] * S0[1][j] + half * S0[0][i] * DS[1][j] + third * DS[0][i] * DS[1][j];
      R pre = 0;
#pragma unroll
      for (int k = 0; k < NW - 1; ++k) {
        pre += DS[2][k] * c;
        R v = fz * pre;
        if (v != R(0)) j_add<R>(g, Jz + base + i + sy * j + sz * k, v);
      }
    }
}

// periodic wrap / deactivation, exactly the sequence of DESIGN.md step 2f
template <class R>
__device__ __forceinline__ bool wrap_axis(R& x, R L, int periodic) {
  if (periodic) {
    if (x < R(0)) x += L;
    if (x >= L) x -= L;
    return false;
  }
  if (!(x >= R(0) && x < L)) {
    x = x < R(0) ? R(0) : nextafter(L, R(0));
    return true;
  }
  return false;
}


}  // namespace pic
