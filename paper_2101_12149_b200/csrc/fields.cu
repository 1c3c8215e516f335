// Yee FDTD update, J guard sum and E/B guard fill (steps 3-5 and the
// guard rules; PAPER.md:78 Yee staggering, PAPER.md:73-77 FillBoundary / SumBoundary).
#include "internal.h"

namespace pic {

namespace {

struct Box3 { int lo[3], n[3]; };

// CKC (ref [12]): the difference of F along axis A at element t, smoothed over the 3x3 transverse
// neighbours: alpha dF(0,0) + beta_ab [dF(+b) + dF(-b)] + beta_ac [dF(+c) + dF(-c)] + gamma [4 corners]
template <class R, int A>
__device__ __forceinline__ R ckc_diff(const Grid<R>& g, const R* __restrict__ F, int t) {
  constexpr int B = (A + 1) % 3, C = (A + 2) % 3;
  const int sa = A == 0 ? 1 : (A == 1 ? g.sy : g.sz);
  const int sb = B == 0 ? 1 : (B == 1 ? g.sy : g.sz);
  const int sc = C == 0 ? 1 : (C == 1 ? g.sy : g.sz);
  auto dF = [&](int o) { return F[t + o + sa] - F[t + o]; };
  return g.ck_a[A] * dF(0) + g.ck_b[A][B] * (dF(sb) + dF(-sb)) + g.ck_b[A][C] * (dF(sc) + dF(-sc)) +
         g.ck_g[A] * (dF(sb + sc) + dF(sb - sc) + dF(-sb + sc) + dF(-sb - sc));
}

// B -= (dt/2) curl E, forward differences (Yee) or CKC-smoothed ones, over the box [lo, lo+n)
template <class R, bool CKC>
__global__ void __launch_bounds__(256) k_push_B(Grid<R> g, Box3 b) {
  int i = blockIdx.x * blockDim.x + threadIdx.x;
  int j = blockIdx.y * blockDim.y + threadIdx.y;
  int k = blockIdx.z;
  if (i >= b.n[0] || j >= b.n[1]) return;
  int t = g.idx(b.lo[0] + i, b.lo[1] + j, b.lo[2] + k);
  const R* __restrict__ Ex = g.F[0];
  const R* __restrict__ Ey = g.F[1];
  const R* __restrict__ Ez = g.F[2];
  if constexpr (CKC) {
    g.F[3][t] -= g.cB[1] * ckc_diff<R, 1>(g, Ez, t) - g.cB[2] * ckc_diff<R, 2>(g, Ey, t);
    g.F[4][t] -= g.cB[2] * ckc_diff<R, 2>(g, Ex, t) - g.cB[0] * ckc_diff<R, 0>(g, Ez, t);
    g.F[5][t] -= g.cB[0] * ckc_diff<R, 0>(g, Ey, t) - g.cB[1] * ckc_diff<R, 1>(g, Ex, t);
  } else {
    R ex = Ex[t], ey = Ey[t], ez = Ez[t];
    g.F[3][t] -= g.cB[1] * (Ez[t + g.sy] - ez) - g.cB[2] * (Ey[t + g.sz] - ey);
    g.F[4][t] -= g.cB[2] * (Ex[t + g.sz] - ex) - g.cB[0] * (Ez[t + 1] - ez);
    g.F[5][t] -= g.cB[0] * (Ey[t + 1] - ey) - g.cB[1] * (Ex[t + g.sy] - ex);
  }
}

// E += dt (c^2 curl B - J/eps0), backward differences
template <class R>
__global__ void __launch_bounds__(256) k_push_E(Grid<R> g, Box3 b) {
  int i = blockIdx.x * blockDim.x + threadIdx.x;
  int j = blockIdx.y * blockDim.y + threadIdx.y;
  int k = blockIdx.z;
  if (i >= b.n[0] || j >= b.n[1]) return;
  int t = g.idx(b.lo[0] + i, b.lo[1] + j, b.lo[2] + k);
  const R* __restrict__ Bx = g.F[3];
  const R* __restrict__ By = g.F[4];
  const R* __restrict__ Bz = g.F[5];
  R bx = Bx[t], by = By[t], bz = Bz[t];
  g.F[0][t] += g.cE[1] * (bz - Bz[t - g.sy]) - g.cE[2] * (by - By[t - g.sz]) - g.cJ * g.J[0][t];
  g.F[1][t] += g.cE[2] * (bx - Bx[t - g.sz]) - g.cE[0] * (bz - Bz[t - 1]) - g.cJ * g.J[1][t];
  g.F[2][t] += g.cE[0] * (by - By[t - 1]) - g.cE[1] * (bx - Bx[t - g.sy]) - g.cJ * g.J[2][t];
}

// The shell of thickness G of a box n0 x n1 x n2 (n >= 2G on every axis), enumerated without the
// interior: 2G full z-planes, then 2G full y-rows of every other plane, then the 2G x-ends of every
// other row. shell_size() points; shell_point() maps a running index to box coordinates.
__host__ __device__ inline int64_t shell_size(int n0, int n1, int n2, int G) {
  return (int64_t)2 * G * n0 * n1 + (int64_t)(n2 - 2 * G) * 2 * G * n0 + (int64_t)(n2 - 2 * G) * (n1 - 2 * G) * 2 * G;
}
__device__ __forceinline__ void shell_point(int64_t idx, int n0, int n1, int n2, int G, int& i, int& j, int& k) {
  const int64_t nA = (int64_t)2 * G * n0 * n1, nB = (int64_t)(n2 - 2 * G) * 2 * G * n0;
  if (idx < nA) {
    i = (int)(idx % n0);
    int64_t r = idx / n0;
    j = (int)(r % n1);
    int kk = (int)(r / n1);                    // 0 .. 2G-1
    k = kk < G ? kk : n2 - 2 * G + kk;
  } else if (idx < nA + nB) {
    idx -= nA;
    i = (int)(idx % n0);
    int64_t r = idx / n0;
    int jj = (int)(r % (2 * G));
    j = jj < G ? jj : n1 - 2 * G + jj;
    k = G + (int)(r / (2 * G));
  } else {
    idx -= nA + nB;
    int ii = (int)(idx % (2 * G));
    i = ii < G ? ii : n0 - 2 * G + ii;
    int64_t r = idx / (2 * G);
    j = G + (int)(r % (n1 - 2 * G));
    k = G + (int)(r / (n1 - 2 * G));
  }
}

// SumBoundary on one periodic box: every valid node within G of a periodic face collects its
// guard images in a fixed order (deterministic, no atomics). Images on a non-periodic axis are
// dropped. One thread per valid node of the shell; three components per thread.
template <class R, bool SHELL>
__global__ void __launch_bounds__(256) k_fold_J(Grid<R> g) {
  int i, j, k;
  if constexpr (SHELL) {   // only the nodes within G of a face (needs N >= 2G)
    const int64_t idx = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (idx >= shell_size(g.N[0], g.N[1], g.N[2], kGuard)) return;
    shell_point(idx, g.N[0], g.N[1], g.N[2], kGuard, i, j, k);
  } else {
    i = blockIdx.x * blockDim.x + threadIdx.x;
    j = blockIdx.y * blockDim.y + threadIdx.y;
    k = blockIdx.z;
    if (i >= g.N[0] || j >= g.N[1]) return;
  }
  const int G = kGuard;
  int c[3] = {i, j, k};
  int lo[3], hi[3];
  bool any = false;
  for (int d = 0; d < 3; ++d) {
    // image shifts s*N with s in [lo,hi]: c - N >= -G  <=>  c >= N-G (image below); c + N < N+G <=> c < G
    lo[d] = (g.periodic[d] && c[d] >= g.N[d] - G) ? -1 : 0;
    hi[d] = (g.periodic[d] && c[d] < G) ? 1 : 0;
    any |= (lo[d] != 0) | (hi[d] != 0);
  }
  if (!any) return;
  int t = g.idx(i, j, k);
  for (int comp = 0; comp < 3; ++comp) {
    R* __restrict__ J = g.J[comp];
    R acc = J[t];
    for (int sc = lo[2]; sc <= hi[2]; ++sc)
      for (int sb = lo[1]; sb <= hi[1]; ++sb)
        for (int sa = lo[0]; sa <= hi[0]; ++sa) {
          if (sa == 0 && sb == 0 && sc == 0) continue;
          acc += J[g.idx(i + sa * g.N[0], j + sb * g.N[1], k + sc * g.N[2])];
        }
    J[t] = acc;
  }
}

// FillBoundary on one periodic box: guard <- periodic image in the valid region. Guards on a
// non-periodic axis are left untouched (they hold zeros). Up to 6 arrays per launch.
template <class R>
struct ArrList { R* a[6]; int n; };

template <class R>
__global__ void __launch_bounds__(256) k_fill_guards(Grid<R> g, ArrList<R> arrs) {
  const int64_t idx = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;   // over the guard shell only
  if (idx >= shell_size(g.P[0], g.P[1], g.P[2], kGuard)) return;
  int i, j, k;
  shell_point(idx, g.P[0], g.P[1], g.P[2], kGuard, i, j, k);
  i -= kGuard; j -= kGuard; k -= kGuard;
  int c[3] = {i, j, k};
  int s[3];
  bool guard = false;
  for (int d = 0; d < 3; ++d) {
    s[d] = c[d];
    if (c[d] < 0 || c[d] >= g.N[d]) {
      if (!g.periodic[d]) return;           // zero guard stays zero
      guard = true;
      s[d] = c[d] < 0 ? c[d] + g.N[d] : c[d] - g.N[d];
      if (s[d] < 0 || s[d] >= g.N[d]) return;   // N < G: cannot happen (checked at create)
    }
  }
  if (!guard) return;
  int dst = g.idx(i, j, k), src = g.idx(s[0], s[1], s[2]);
  for (int a = 0; a < arrs.n; ++a) arrs.a[a][dst] = arrs.a[a][src];
}

template <class R>
__global__ void __launch_bounds__(256) k_pack(Grid<R> g, const R* __restrict__ src, R* __restrict__ dst) {
  int i = blockIdx.x * blockDim.x + threadIdx.x;
  int j = blockIdx.y * blockDim.y + threadIdx.y;
  int k = blockIdx.z;
  if (i >= g.N[0] || j >= g.N[1]) return;
  dst[g.idx(i, j, k)] = src[(size_t)i + (size_t)g.N[0] * ((size_t)j + (size_t)g.N[1] * k)];
}

template <class R>
__global__ void __launch_bounds__(256) k_unpack(Grid<R> g, const R* __restrict__ src, R* __restrict__ dst) {
  int i = blockIdx.x * blockDim.x + threadIdx.x;
  int j = blockIdx.y * blockDim.y + threadIdx.y;
  int k = blockIdx.z;
  if (i >= g.N[0] || j >= g.N[1]) return;
  dst[(size_t)i + (size_t)g.N[0] * ((size_t)j + (size_t)g.N[1] * k)] = src[g.idx(i, j, k)];
}

inline dim3 blk() { return dim3(64, 4, 1); }
inline dim3 grd(int nx, int ny, int nz) { return dim3((nx + 63) / 64, (ny + 3) / 4, nz); }

}  // namespace

template <class R>
void launch_push_B(const Grid<R>& g, const int lo[3], const int hi[3], Ctx& c) {
  Box3 b;
  for (int d = 0; d < 3; ++d) { b.lo[d] = lo[d]; b.n[d] = hi[d] - lo[d]; }
  if (g.solver == 1) k_push_B<R, true><<<grd(b.n[0], b.n[1], b.n[2]), blk(), 0, c.stream>>>(g, b);
  else k_push_B<R, false><<<grd(b.n[0], b.n[1], b.n[2]), blk(), 0, c.stream>>>(g, b);
  c.launches++;
}
template <class R>
void launch_push_E(const Grid<R>& g, const int lo[3], const int hi[3], Ctx& c) {
  Box3 b;
  for (int d = 0; d < 3; ++d) { b.lo[d] = lo[d]; b.n[d] = hi[d] - lo[d]; }
  k_push_E<R><<<grd(b.n[0], b.n[1], b.n[2]), blk(), 0, c.stream>>>(g, b);
  c.launches++;
}
// deterministic deposition: the two fixed-point parts of every J element -> J (common.cuh, j_add)
template <class R>
__global__ void __launch_bounds__(256) k_fix_to_J(Grid<R> g, int64_t n) {
  const int64_t t = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (t >= n) return;
  g.J[0][t] = (R)((double)g.Jfix[0][t] * g.fix_inv[0] + (double)g.Jfix[1][t] * g.fix_inv[1]);
}
template <class R>
void launch_fix_to_J(const Grid<R>& g, Ctx& c) {
  const int64_t n = 3 * g.padded_total();   // the three J arrays are one allocation
  k_fix_to_J<R><<<(unsigned)((n + 255) / 256), 256, 0, c.stream>>>(g, n);
  c.launches++;
}
template <class R>
void launch_fold_J(const Grid<R>& g, Ctx& c) {
  if (g.N[0] >= 2 * kGuard && g.N[1] >= 2 * kGuard && g.N[2] >= 2 * kGuard) {
    const int64_t n = shell_size(g.N[0], g.N[1], g.N[2], kGuard);
    k_fold_J<R, true><<<(unsigned)((n + 255) / 256), 256, 0, c.stream>>>(g);
  } else {
    k_fold_J<R, false><<<grd(g.N[0], g.N[1], g.N[2]), blk(), 0, c.stream>>>(g);
  }
  c.launches++;
}
template <class R>
void launch_fill_guards(const Grid<R>& g, R* const* arrays, int narr, Ctx& c) {
  ArrList<R> l;
  l.n = narr;
  for (int a = 0; a < 6; ++a) l.a[a] = a < narr ? arrays[a] : nullptr;
  const int64_t n = shell_size(g.P[0], g.P[1], g.P[2], kGuard);
  k_fill_guards<R><<<(unsigned)((n + 255) / 256), 256, 0, c.stream>>>(g, l);
  c.launches++;
}
template <class R>
void launch_pack(const Grid<R>& g, const R* src, R* dst, Ctx& c) {
  k_pack<R><<<grd(g.N[0], g.N[1], g.N[2]), blk(), 0, c.stream>>>(g, src, dst);
  c.launches++;
}
template <class R>
void launch_unpack(const Grid<R>& g, const R* src, R* dst, Ctx& c) {
  k_unpack<R><<<grd(g.N[0], g.N[1], g.N[2]), blk(), 0, c.stream>>>(g, src, dst);
  c.launches++;
}

#define INST(R)                                                                         \
  template void launch_push_B<R>(const Grid<R>&, const int*, const int*, Ctx&);         \
  template void launch_push_E<R>(const Grid<R>&, const int*, const int*, Ctx&);         \
  template void launch_fold_J<R>(const Grid<R>&, Ctx&);                                 \
  template void launch_fix_to_J<R>(const Grid<R>&, Ctx&);                               \
  template void launch_fill_guards<R>(const Grid<R>&, R* const*, int, Ctx&);            \
  template void launch_pack<R>(const Grid<R>&, const R*, R*, Ctx&);                     \
  template void launch_unpack<R>(const Grid<R>&, const R*, R*, Ctx&);
INST(double)
INST(float)
#undef INST

}  // namespace pic
