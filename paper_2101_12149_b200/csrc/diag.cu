// Input validation and diagnostics reductions (support, not on the hot path; PAPER.md:98-102
// §2.6: several reductions in one launch). All accumulators are fp64.
#include <algorithm>

#include "internal.h"

namespace pic {

namespace {

__device__ __forceinline__ double warp_sum(double v) {
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
  return v;
}
__device__ __forceinline__ double warp_max(double v) {
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) v = fmax(v, __shfl_xor_sync(0xffffffffu, v, o));
  return v;
}
// non-negative doubles order like their bit patterns
__device__ __forceinline__ void atomic_max_nonneg(double* p, double v) {
  atomicMax((unsigned long long*)p, (unsigned long long)__double_as_longlong(v));
}

// flags[0] |= non-finite value seen, flags[1] |= position outside [0, L)
template <class R>
__global__ void __launch_bounds__(256) k_validate_particles(Grid<R> g, Particles<R> p, int* flags) {
  int64_t t = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (t >= p.n) return;
  R v[7] = {p.x[t], p.y[t], p.z[t], p.ux[t], p.uy[t], p.uz[t], p.w[t]};
  bool bad = false;
#pragma unroll
  for (int a = 0; a < 7; ++a) bad |= !isfinite(v[a]);
  bool out = false;
#pragma unroll
  for (int d = 0; d < 3; ++d) out |= !(v[d] >= R(0) && v[d] < g.L[d]);
  if (bad) atomicOr(&flags[0], 1);
  else if (out) atomicOr(&flags[1], 1);
}

template <class R>
__global__ void __launch_bounds__(256) k_validate_array(const R* __restrict__ a, int64_t n, int* flags) {
  int64_t t = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (t < n && !isfinite(a[t])) atomicOr(&flags[0], 1);
}

template <class R>
__global__ void __launch_bounds__(256) k_field_energy(Grid<R> g, double* out2) {
  int i = blockIdx.x * blockDim.x + threadIdx.x;
  int j = blockIdx.y * blockDim.y + threadIdx.y;
  int k = blockIdx.z;
  double e2 = 0, b2 = 0;
  if (i < g.N[0] && j < g.N[1]) {
    int t = g.idx(i, j, k);
#pragma unroll
    for (int c = 0; c < 3; ++c) {
      double e = (double)g.F[c][t], b = (double)g.F[3 + c][t];
      e2 += e * e;
      b2 += b * b;
    }
  }
  e2 = warp_sum(e2);
  b2 = warp_sum(b2);
  if (((threadIdx.x + blockDim.x * threadIdx.y) & 31) == 0) {
    atomicAdd(&out2[0], e2);
    atomicAdd(&out2[1], b2);
  }
}

template <class R>
__global__ void __launch_bounds__(256) k_particle_sums(Particles<R> p, double q, double m, double* out2) {
  int64_t t = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  double ke = 0, ch = 0;
  if (t < p.n) {
    double ux = p.ux[t], uy = p.uy[t], uz = p.uz[t], w = p.w[t];
    double a = (ux * ux + uy * uy + uz * uz) / (kC * kC);
    double gm1 = a / (1.0 + sqrt(1.0 + a));
    ke = w * m * kC * kC * gm1;
    ch = q * w;
  }
  ke = warp_sum(ke);
  ch = warp_sum(ch);
  if ((threadIdx.x & 31) == 0) {
    atomicAdd(&out2[0], ke);
    atomicAdd(&out2[1], ch);
  }
}

__device__ __forceinline__ int wrap_idx(int i, int N, int periodic) {
  if (periodic) {
    i %= N;
    return i < 0 ? i + N : i;
  }
  return (i < 0 || i >= N) ? -1 : i;
}

// nodal charge density on the valid region (indices wrapped), fp64 atomics
template <class R, int ORDER>
__global__ void __launch_bounds__(128) k_rho(Grid<R> g, Particles<R> p, double q, double* rho) {
  int64_t t = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (t >= p.n) return;
  R w[3][ORDER + 1];
  int l[3];
  R pos[3] = {p.x[t], p.y[t], p.z[t]};
#pragma unroll
  for (int d = 0; d < 3; ++d) l[d] = shape<R, ORDER>(mul_rn(pos[d], g.inv_dx[d]), w[d]);
  double inv_dv = (double)g.inv_dx[0] * (double)g.inv_dx[1] * (double)g.inv_dx[2];
  double qw = q * (double)p.w[t] * inv_dv;
#pragma unroll
  for (int c = 0; c <= ORDER; ++c)
#pragma unroll
    for (int b = 0; b <= ORDER; ++b)
#pragma unroll
      for (int a = 0; a <= ORDER; ++a) {
        int i = wrap_idx(l[0] + a, g.N[0], g.periodic[0]);
        int j = wrap_idx(l[1] + b, g.N[1], g.periodic[1]);
        int k = wrap_idx(l[2] + c, g.N[2], g.periodic[2]);
        if (i >= 0 && j >= 0 && k >= 0)
          atomicAdd(&rho[(size_t)i + (size_t)g.N[0] * ((size_t)j + (size_t)g.N[1] * k)],
                    qw * (double)(w[0][a] * w[1][b] * w[2][c]));
      }
}

template <class R>
__global__ void __launch_bounds__(256) k_gauss(Grid<R> g, const double* __restrict__ rho, double* out2) {
  int i = blockIdx.x * blockDim.x + threadIdx.x;
  int j = blockIdx.y * blockDim.y + threadIdx.y;
  int k = blockIdx.z;
  double res = 0, rm = 0;
  if (i < g.N[0] && j < g.N[1]) {
    int t = g.idx(i, j, k);
    double div = ((double)g.F[0][t] - (double)g.F[0][t - 1]) * (double)g.inv_dx[0] +
                 ((double)g.F[1][t] - (double)g.F[1][t - g.sy]) * (double)g.inv_dx[1] +
                 ((double)g.F[2][t] - (double)g.F[2][t - g.sz]) * (double)g.inv_dx[2];
    double r = rho[(size_t)i + (size_t)g.N[0] * ((size_t)j + (size_t)g.N[1] * k)] / kEps0;
    res = fabs(div - r);
    rm = fabs(r);
  }
  res = warp_max(res);
  rm = warp_max(rm);
  if (((threadIdx.x + blockDim.x * threadIdx.y) & 31) == 0) {
    atomic_max_nonneg(&out2[0], res);
    atomic_max_nonneg(&out2[1], rm);
  }
}

inline dim3 blk() { return dim3(64, 4, 1); }
inline dim3 grd(int nx, int ny, int nz) { return dim3((nx + 63) / 64, (ny + 3) / 4, nz); }

}  // namespace

template <class R>
void launch_validate_particles(const Grid<R>& g, const Particles<R>& p, int* flags, Ctx& c) {
  if (p.n == 0) return;
  k_validate_particles<R><<<(unsigned)((p.n + 255) / 256), 256, 0, c.stream>>>(g, p, flags);
  c.launches++;
}
template <class R>
void launch_validate_array(const R* a, int64_t n, int* flags, Ctx& c) {
  if (n == 0) return;
  k_validate_array<R><<<(unsigned)((n + 255) / 256), 256, 0, c.stream>>>(a, n, flags);
  c.launches++;
}
// max |a| into *out (non-negative doubles order like their bit patterns, so an integer atomicMax does it
// exactly and independently of the order of arrival)
template <class R>
__global__ void __launch_bounds__(256) k_max_abs(const R* __restrict__ a, int64_t n, double* out) {
  double m = 0.0;
  for (int64_t t = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; t < n; t += (int64_t)gridDim.x * blockDim.x)
    m = fmax(m, fabs((double)a[t]));
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) m = fmax(m, __shfl_xor_sync(0xffffffffu, m, o));
  if ((threadIdx.x & 31) == 0) atomicMax(reinterpret_cast<unsigned long long*>(out), (unsigned long long)__double_as_longlong(m));
}
template <class R>
void launch_max_abs(const R* a, int64_t n, double* out1, Ctx& c) {
  if (n == 0) return;
  const int64_t nb = std::min<int64_t>((n + 255) / 256, (int64_t)c.sm_count * 16);
  k_max_abs<R><<<(unsigned)nb, 256, 0, c.stream>>>(a, n, out1);
  c.launches++;
}
template <class R>
void launch_field_energy(const Grid<R>& g, double* out2, Ctx& c) {
  k_field_energy<R><<<grd(g.N[0], g.N[1], g.N[2]), blk(), 0, c.stream>>>(g, out2);
  c.launches++;
}
template <class R>
void launch_particle_sums(const Particles<R>& p, double q, double m, double* out2, Ctx& c) {
  if (p.n == 0) return;
  k_particle_sums<R><<<(unsigned)((p.n + 255) / 256), 256, 0, c.stream>>>(p, q, m, out2);
  c.launches++;
}
template <class R>
void launch_rho(const Grid<R>& g, const Particles<R>& p, int order, double q, double* rho, Ctx& c) {
  if (p.n == 0) return;
  unsigned nb = (unsigned)((p.n + 127) / 128);
  if (order == 1) k_rho<R, 1><<<nb, 128, 0, c.stream>>>(g, p, q, rho);
  else if (order == 2) k_rho<R, 2><<<nb, 128, 0, c.stream>>>(g, p, q, rho);
  else k_rho<R, 3><<<nb, 128, 0, c.stream>>>(g, p, q, rho);
  c.launches++;
}
template <class R>
void launch_gauss(const Grid<R>& g, const double* rho, double* out2, Ctx& c) {
  k_gauss<R><<<grd(g.N[0], g.N[1], g.N[2]), blk(), 0, c.stream>>>(g, rho, out2);
  c.launches++;
}

#define INST(R)                                                                                    \
  template void launch_validate_particles<R>(const Grid<R>&, const Particles<R>&, int*, Ctx&);     \
  template void launch_validate_array<R>(const R*, int64_t, int*, Ctx&);                           \
  template void launch_max_abs<R>(const R*, int64_t, double*, Ctx&);                               \
  template void launch_field_energy<R>(const Grid<R>&, double*, Ctx&);                             \
  template void launch_particle_sums<R>(const Particles<R>&, double, double, double*, Ctx&);       \
  template void launch_rho<R>(const Grid<R>&, const Particles<R>&, int, double, double*, Ctx&);    \
  template void launch_gauss<R>(const Grid<R>&, const double*, double*, Ctx&);
INST(double)
INST(float)
#undef INST

}  // namespace pic
