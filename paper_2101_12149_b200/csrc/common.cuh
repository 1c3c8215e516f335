// Shared device-side definitions of the CUDA path (sm_100a). Not used by oracle/.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

namespace pic {

// CODATA 2018.
constexpr double kC = 299792458.0;
constexpr double kEps0 = 8.8541878128e-12;

constexpr int kGuard = 4;  // guard cells per side

// Field storage: every component is a padded box (N+2G)^3, x fastest; (i,j,k) in [-G, N+G).
template <class R>
struct Grid {
  int N[3];
  int P[3];          // padded extents
  int sy, sz;        // strides of j and k in elements (sx = 1)
  int org;           // linear offset of node (0,0,0)
  int periodic[3];
  int pusher;        // PIC_PUSHER_*
  int gather_mode;   // PIC_GATHER_*
  int solver;        // PIC_SOLVER_*
  R ck_a[3], ck_b[3][3], ck_g[3];   // CKC weights alpha_a, beta_ab, gamma_a
  R inv_dx[3], L[3], cB[3], cE[3], cJ, inv_c2, dt;
  R* F[6];           // Ex Ey Ez Bx By Bz
  R* J[3];
  // deterministic deposition (PIC_DEPOSIT order-free sums): every contribution to J is
  // split into two 64-bit fixed-point parts that are added with INTEGER reductions (exact, hence independent
  // of the order in which warps arrive); Jfix[0] / Jfix[1] shadow the three J arrays (same offsets)
  long long* Jfix[2];
  double fix_scale[2];   // 2^e_hi, 2^e_lo (e_lo = e_hi + 40); 0 = mode off
  double fix_inv[2];
  __host__ __device__ __forceinline__ int idx(int i, int j, int k) const { return org + i + sy * j + sz * k; }
  __host__ __device__ __forceinline__ int64_t padded_total() const { return (int64_t)P[0] * P[1] * P[2]; }
};

// One species' particle arrays (structure of arrays).
template <class R>
struct Particles {
  R *x, *y, *z, *ux, *uy, *uz, *w;
  int64_t* id;
  int64_t n;
  R kq;      // q*dt/(2m)
  R jf[3];   // q/(dt*dx_a*dx_b)
};

struct TileSpec {
  int T[3];      // cells per tile
  int nt[3];     // tiles per axis
  int tvol;      // cells per tile
  int key_mode;  // 0 tile-major cell key, 1 tile only
};

// ------------------------------------------------------------------ rounded arithmetic
// Operations the compiler may neither contract into an FMA nor reassociate. mul_rn: the one rounded
// multiply of the sort rule and of every normalised coordinate xi = x * inv_dx.
// sub_rn: difference of two ROUNDED values (DS = S1 - S0 cancels to roundoff for a slow particle).
// In fp32 the whole chain position -> weights -> gathered field -> momentum -> new position is written
// with them in the operation order of the method's statement (left to
// right), so that x_new and u_new come out bit for bit what that statement gives in IEEE single
// precision: one fp32 ulp of a position is 1e-3 of a step's displacement at 128 cells, and the
// deposit's DS = S1 - S0 would otherwise carry that into J.
__device__ __forceinline__ double mul_rn(double a, double b) { return __dmul_rn(a, b); }
__device__ __forceinline__ float mul_rn(float a, float b) { return __fmul_rn(a, b); }
__device__ __forceinline__ double sub_rn(double a, double b) { return __dsub_rn(a, b); }
__device__ __forceinline__ float sub_rn(float a, float b) { return __fsub_rn(a, b); }
__device__ __forceinline__ double add_rn(double a, double b) { return __dadd_rn(a, b); }
__device__ __forceinline__ float add_rn(float a, float b) { return __fadd_rn(a, b); }
__device__ __forceinline__ double div_rn(double a, double b) { return __ddiv_rn(a, b); }
__device__ __forceinline__ float div_rn(float a, float b) { return __fdiv_rn(a, b); }
__device__ __forceinline__ double sqrt_rn(double a) { return __dsqrt_rn(a); }
__device__ __forceinline__ float sqrt_rn(float a) { return __fsqrt_rn(a); }
// fp32: statement order, every operation rounded; fp64: the compiler's contractions are welcome
// (they only add accuracy, and 1e-12 leaves room for them)
template <class R> constexpr bool kStatementOrder = sizeof(R) == 4;

// ------------------------------------------------------------------ shape factors
// B-spline weights of order n at normalised coordinate xi; returns the leftmost node index.
template <class R, int ORDER>
__device__ __forceinline__ int shape(R xi, R* w) {
  if constexpr (kStatementOrder<R>) {
    const R h = R(0.5);
    if constexpr (ORDER == 1) {
      R m = floor(xi);
      R d = sub_rn(xi, m);
      w[0] = sub_rn(R(1), d);
      w[1] = d;
      return (int)m;
    } else if constexpr (ORDER == 2) {
      R m = floor(add_rn(xi, h));
      R d = sub_rn(xi, m);
      R a = sub_rn(h, d), b = add_rn(h, d);
      w[0] = mul_rn(mul_rn(h, a), a);
      w[1] = sub_rn(R(0.75), mul_rn(d, d));
      w[2] = mul_rn(mul_rn(h, b), b);
      return (int)m - 1;
    } else {
      R m = floor(xi);
      R d = sub_rn(xi, m);
      R e = sub_rn(R(1), d);
      w[0] = div_rn(mul_rn(mul_rn(e, e), e), R(6));
      w[1] = div_rn(add_rn(sub_rn(R(4), mul_rn(mul_rn(R(6), d), d)), mul_rn(mul_rn(mul_rn(R(3), d), d), d)), R(6));
      w[2] = div_rn(add_rn(sub_rn(R(4), mul_rn(mul_rn(R(6), e), e)), mul_rn(mul_rn(mul_rn(R(3), e), e), e)), R(6));
      w[3] = div_rn(mul_rn(mul_rn(d, d), d), R(6));
      return (int)m - 1;
    }
  } else if constexpr (ORDER == 1) {
    R m = floor(xi);
    R d = xi - m;
    w[0] = R(1) - d;
    w[1] = d;
    return (int)m;
  } else if constexpr (ORDER == 2) {
    R m = floor(xi + R(0.5));
    R d = xi - m;
    R a = R(0.5) - d, b = R(0.5) + d;
    w[0] = R(0.5) * a * a;
    w[1] = R(0.75) - d * d;
    w[2] = R(0.5) * b * b;
    return (int)m - 1;
  } else {
    R m = floor(xi);
    R d = xi - m;
    R e = R(1) - d;
    const R s = R(1) / R(6);
    w[0] = e * e * e * s;
    w[1] = (R(4) - R(6) * d * d + R(3) * d * d * d) * s;
    w[2] = (R(4) - R(6) * e * e + R(3) * e * e * e) * s;
    w[3] = d * d * d * s;
    return (int)m - 1;
  }
}

// Galerkin gather: order ORDER-1 at a staggered coordinate, returned on ORDER+1 slots
// (the last weight is zero) so that it drops into the loops of the uniform gather unchanged.
template <class R, int ORDER>
__device__ __forceinline__ int shape_lowered(R xi, R* w) {
  w[ORDER] = R(0);
  if constexpr (ORDER == 1) {            // order 0: nearest grid point
    w[0] = R(1);
    return (int)floor(add_rn(xi, R(0.5)));
  } else {
    return shape<R, ORDER - 1>(xi, w);
  }
}

template <class R>
__device__ __forceinline__ int cell_of(R x, R inv_dx, int N) {
  int c = (int)floor(mul_rn(x, inv_dx));
  return min(max(c, 0), N - 1);
}

// reduction without return value (RED.E.ADD.F64 / .F32 at L2)
__device__ __forceinline__ void red_add(double* p, double v) { atomicAdd(p, v); }
__device__ __forceinline__ void red_add(float* p, float v) { atomicAdd(p, v); }

// One contribution v to the J element at p (p points into g.J[0..2], which are one allocation). Default: a
// floating-point reduction at L2, whose result depends on the order of arrival. Deterministic mode: v is
// split into hi = rint(v 2^e_hi) and lo = rint((v - hi 2^-e_hi) 2^e_lo), both added as 64-bit integers;
// integer addition is associative, so J comes out bit-identical whatever the order (k_fix_to_J converts).
// 2^e_hi is chosen from a bound no node can exceed (pic_api.cu), the low part carries 40 more bits.
// DET: 0 = floating-point reduction, 1 = fixed point, -1 = whichever the grid says (run-time test; the hot
// kernels are compiled for both and never pay for it).
template <class R, int DET = -1>
__device__ __forceinline__ void j_add(const Grid<R>& g, R* p, R v) {
  if (DET == 1 || (DET == -1 && g.fix_scale[0] != 0.0)) {
    const long long off = p - g.J[0];
    const double hi = rint((double)v * g.fix_scale[0]);
    const double lo = rint(((double)v - hi * g.fix_inv[0]) * g.fix_scale[1]);
    atomicAdd(reinterpret_cast<unsigned long long*>(g.Jfix[0] + off), (unsigned long long)(long long)hi);
    atomicAdd(reinterpret_cast<unsigned long long*>(g.Jfix[1] + off), (unsigned long long)(long long)lo);
  } else {
    red_add(p, v);
  }
}

}  // namespace pic
