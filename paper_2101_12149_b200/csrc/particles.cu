// Particle kernels: fused field gather + relativistic Boris push, and
// Esirkepov current deposition in two designs that compute the same sums:
//   GLOBAL  one thread per particle, gather+push+deposit fused, one global reduction per
//           particle-node (the paper's GPU design);
//   COOP    gather+push kernel (one thread per particle), then a warp-cooperative deposition:
//           a warp walks its cell-sorted particles, lanes own the (j,k) nodes of the cell's
//           window, x runs along registers; sums stay in registers for a whole run of cells
//           along x and reach memory once per node (fp64/fp32 reductions at L2).
// PAPER.md:114 (fused gather+push, no per-particle E/B), PAPER.md:167-175 (deposition),
// ref [8] Esirkepov PAPER.md:301.
#include <climits>

#include <algorithm>

#include "internal.h"
#include "particle_math.cuh"

namespace pic {

namespace {

template <class R, int ORDER>
__global__ void __launch_bounds__(128) k_particles_global(Grid<R> g, Particles<R> p, unsigned long long* deactivated) {
  int64_t t = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (t >= p.n) return;
  R x0[3] = {p.x[t], p.y[t], p.z[t]};
  R u[3] = {p.ux[t], p.uy[t], p.uz[t]};
  R w = p.w[t];
  R E[3], B[3];
  gather6<R, ORDER>(g, x0[0], x0[1], x0[2], E, B);
  push_momentum<R>(g.pusher, p.kq, g.inv_c2, E, B, u);
  R x1[3];
  advance<R>(g.dt, g.inv_c2, x0, u, x1);
  deposit_global<R, ORDER>(g, p.jf, w, x0, x1);
  bool out = false;
#pragma unroll
  for (int d = 0; d < 3; ++d) out |= wrap_axis<R>(x1[d], g.L[d], g.periodic[d]);
  if (out) {
    if (w != R(0)) atomicAdd(deactivated, 1ull);
    p.w[t] = R(0);
  }
  p.x[t] = x1[0]; p.y[t] = x1[1]; p.z[t] = x1[2];
  p.ux[t] = u[0]; p.uy[t] = u[1]; p.uz[t] = u[2];
}

// ------------------------------------------------------------------ COOP, kernel 1: gather + push
// Reads x^n, u^{n-1/2}; writes u^{n+1/2} in place and the UNWRAPPED new position into `xn`.
template <class R, int ORDER>
__global__ void __launch_bounds__(128) k_push(Grid<R> g, Particles<R> p, R* __restrict__ xn, R* __restrict__ yn,
                                              R* __restrict__ zn) {
  int64_t t = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (t >= p.n) return;
  R x0[3] = {p.x[t], p.y[t], p.z[t]};
  R u[3] = {p.ux[t], p.uy[t], p.uz[t]};
  R E[3], B[3];
  gather6<R, ORDER>(g, x0[0], x0[1], x0[2], E, B);
  push_momentum<R>(g.pusher, p.kq, g.inv_c2, E, B, u);
  R x1[3];
  advance<R>(g.dt, g.inv_c2, x0, u, x1);
  xn[t] = x1[0]; yn[t] = x1[1]; zn[t] = x1[2];
  p.ux[t] = u[0]; p.uy[t] = u[1]; p.uz[t] = u[2];
}

// ------------------------------------------------------------------ COOP, kernel 2: deposition
template <class R>
struct alignas(2 * sizeof(R)) Pair { R a, b; };

template <int ORDER>
struct Win {
  static constexpr int NW = ORDER == 1 ? 4 : 6;   // nodes per axis of the window fixed to a CELL
  static constexpr int BL = ORDER == 1 ? 1 : 2;   // window base = cell - BL
  static constexpr int REC = 9 * NW + (NW == 4 ? 2 : 0);   // record stride: conflict-free stores
  // record layout (elements): {A_x,B_x}[NW] | {S0_y,DS_y}[NW] | {S0_z,DS_z}[NW] | PX[NW] | PY[NW] | PZ[NW]
  static constexpr int oABX = 0, oY = 2 * NW, oZ = 4 * NW, oPX = 6 * NW, oPY = 7 * NW, oPZ = 8 * NW;
};

constexpr int kCoopWarps = 4;        // warps per CTA
constexpr int kCoopChunk = 512;      // consecutive particles walked by one warp

// Per axis: old/new weights placed on the cell's window, DS, A = S0 + DS/2, B = S0/2 + DS/3 and
// the running sum of DS (Esirkepov: W_x = DS_x (S0_z A_y + DS_z B_y), J_x = -q w/(dt dy dz) cumsum_x W_x, cyclic).
template <class R, int ORDER>
__device__ __forceinline__ void axis_record(R xi0, R xi1, int N, int& cell, R* S0, R* DS, bool& edge) {
  constexpr int NW = Win<ORDER>::NW, BL = Win<ORDER>::BL;
  R w0[ORDER + 1], w1[ORDER + 1];
  int l0 = shape<R, ORDER>(xi0, w0);
  int l1 = shape<R, ORDER>(xi1, w1);
  int c = ORDER == 2 ? (int)floor(xi0) : (ORDER == 1 ? l0 : l0 + 1);
  c = min(max(c, 0), N);
  int so0 = l0 - (c - BL), sl1 = l1 - (c - BL);
  R S1[NW];
#pragma unroll
  for (int i = 0; i < NW; ++i) {
    R a = 0, b = 0;
#pragma unroll
    for (int k = 0; k <= ORDER; ++k) {
      a = (i == so0 + k) ? w0[k] : a;
      b = (i == sl1 + k) ? w1[k] : b;
    }
    S0[i] = a;
    S1[i] = b;
    DS[i] = sub_rn(b, a);
  }
  edge = (S0[0] != R(0)) | (S1[0] != R(0)) | (S0[NW - 1] != R(0)) | (S1[NW - 1] != R(0));
  cell = c;
}

template <class R, int ORDER>
__global__ void __launch_bounds__(kCoopWarps * 32) k_deposit_coop(Grid<R> g, Particles<R> p, R* __restrict__ xn,
                                                                  R* __restrict__ yn, R* __restrict__ zn,
                                                                  const int32_t* __restrict__ cell_sorted,
                                                                  int32_t* __restrict__ stray_list,
                                                                  unsigned int* __restrict__ stray_count,
                                                                  unsigned long long* deactivated) {
  using W = Win<ORDER>;
  constexpr int NW = W::NW, BL = W::BL, REC = W::REC;
  extern __shared__ __align__(16) unsigned char smem_raw[];
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  R* rec = reinterpret_cast<R*>(smem_raw) + (size_t)warp * 32 * REC;
  // lane -> (j,k) of the window; the 6x6 window has 36 pairs: its 4 corners are never needed by
  // the particles this kernel accepts (a corner needs a cell change in y AND z; those go to the list)
  int pair = lane;
  bool lane_on = true;
  if (NW == 6) pair = lane < 4 ? lane + 1 : (lane < 28 ? lane + 2 : lane + 3);
  else lane_on = lane < NW * NW;
  const int j = lane_on ? pair / NW : 0, k = lane_on ? pair % NW : 0;
  const int off_jk = g.sy * j + g.sz * k;
  const R half = R(0.5), third = R(1) / R(3);

  R ax[NW - 1], ay[NW], az[NW];
#pragma unroll
  for (int i = 0; i < NW; ++i) { ay[i] = 0; az[i] = 0; if (i < NW - 1) ax[i] = 0; }
  int cur_ib = INT_MIN;    // window base index of the run being accumulated

  auto flush_all = [&]() {
    if (cur_ib == INT_MIN || !lane_on) return;
    R* jx = g.J[0] + cur_ib + off_jk;
    R* jy = g.J[1] + cur_ib + off_jk;
    R* jz = g.J[2] + cur_ib + off_jk;
#pragma unroll
    for (int i = 0; i < NW; ++i) {
      if (i < NW - 1 && ax[i] != R(0)) j_add<R>(g, jx + i, ax[i]);
      if (ay[i] != R(0)) j_add<R>(g, jy + i, ay[i]);
      if (az[i] != R(0)) j_add<R>(g, jz + i, az[i]);
    }
  };
  auto zero_all = [&]() {
#pragma unroll
    for (int i = 0; i < NW; ++i) { ay[i] = 0; az[i] = 0; if (i < NW - 1) ax[i] = 0; }
  };
  auto shift_one = [&]() {   // the run moves one cell up in x: x-slot 0 is complete
    if (lane_on) {
      if (ax[0] != R(0)) j_add<R>(g, g.J[0] + cur_ib + off_jk, ax[0]);
      if (ay[0] != R(0)) j_add<R>(g, g.J[1] + cur_ib + off_jk, ay[0]);
      if (az[0] != R(0)) j_add<R>(g, g.J[2] + cur_ib + off_jk, az[0]);
    }
#pragma unroll
    for (int i = 0; i < NW - 1; ++i) { ay[i] = ay[i + 1]; az[i] = az[i + 1]; if (i < NW - 2) ax[i] = ax[i + 1]; }
    ay[NW - 1] = 0; az[NW - 1] = 0; ax[NW - 2] = 0;
    cur_ib += 1;
  };

  // a warp walks kCoopChunk consecutive particles
  const int64_t wg = (int64_t)blockIdx.x * kCoopWarps + warp;
  const int64_t begin = wg * kCoopChunk;
  const int64_t end = min(p.n, begin + kCoopChunk);
  for (int64_t b0 = begin; b0 < end; b0 += 32) {
    const bool valid = b0 + lane < end;
    const int64_t t = valid ? b0 + lane : 0;
    bool elig = false;
    int ib = 0;
    R x1[3] = {0, 0, 0};
    R w = 0;
    if (valid) {
      R x0[3] = {p.x[t], p.y[t], p.z[t]};
      x1[0] = xn[t]; x1[1] = yn[t]; x1[2] = zn[t];
      w = p.w[t];
      R S0[3][NW], DS[3][NW];
      int c[3];
      bool edge[3];
#pragma unroll
      for (int d = 0; d < 3; ++d)
        axis_record<R, ORDER>(mul_rn(x0[d], g.inv_dx[d]), mul_rn(x1[d], g.inv_dx[d]), g.N[d], c[d], S0[d], DS[d], edge[d]);
      elig = cell_sorted == nullptr || cell_sorted[t] == c[0] + g.N[0] * (c[1] + g.N[1] * c[2]);
      if (NW * NW > 32) elig &= !(edge[1] && edge[2]);
      if (elig) {
        ib = g.idx(c[0] - BL, c[1] - BL, c[2] - BL);
        R* r = rec + lane * REC;
        const R fx = -(w * p.jf[0]), fy = -(w * p.jf[1]), fz = -(w * p.jf[2]);
        R px = 0, py = 0, pz = 0;
#pragma unroll
        for (int i = 0; i < NW; ++i) {
          Pair<R> ab{S0[0][i] + half * DS[0][i], half * S0[0][i] + third * DS[0][i]};
          *reinterpret_cast<Pair<R>*>(r + W::oABX + 2 * i) = ab;
          *reinterpret_cast<Pair<R>*>(r + W::oY + 2 * i) = Pair<R>{S0[1][i], DS[1][i]};
          *reinterpret_cast<Pair<R>*>(r + W::oZ + 2 * i) = Pair<R>{S0[2][i], DS[2][i]};
          px += DS[0][i]; py += DS[1][i]; pz += DS[2][i];
          r[W::oPX + i] = fx * px;
          r[W::oPY + i] = fy * py;
          r[W::oPZ + i] = fz * pz;
        }
      }
    }
    __syncwarp();
    unsigned m = __ballot_sync(0xffffffffu, elig);
    while (m) {
      const int q = __ffs(m) - 1;
      m &= m - 1;
      const int ibq = __shfl_sync(0xffffffffu, ib, q);
      if (ibq != cur_ib) {
        const int s = ibq - cur_ib;
        if (cur_ib != INT_MIN && s > 0 && s < NW) {
          for (int e = 0; e < s; ++e) shift_one();
        } else {
          flush_all();
          zero_all();
          cur_ib = ibq;
        }
      }
      const R* r = rec + q * REC;
      const Pair<R> yv = *reinterpret_cast<const Pair<R>*>(r + W::oY + 2 * j);
      const Pair<R> zv = *reinterpret_cast<const Pair<R>*>(r + W::oZ + 2 * k);
      const R py = r[W::oPY + j], pz = r[W::oPZ + k];
      const R cx = zv.a * (yv.a + half * yv.b) + zv.b * (half * yv.a + third * yv.b);
      const R q1 = py * zv.a, q2 = py * zv.b;
      const R r1 = pz * yv.a, r2 = pz * yv.b;
#pragma unroll
      for (int i = 0; i < NW; ++i) {
        const Pair<R> ab = *reinterpret_cast<const Pair<R>*>(r + W::oABX + 2 * i);
        if (i < NW - 1) ax[i] += cx * r[W::oPX + i];
        ay[i] += q1 * ab.a + q2 * ab.b;
        az[i] += r1 * ab.a + r2 * ab.b;
      }
    }
    __syncwarp();
    // particles deposited here are finished: wrap and store; the others go to the list untouched
    const bool stray = valid && !elig;
    const unsigned sm = __ballot_sync(0xffffffffu, stray);
    if (sm) {
      unsigned base = 0;
      if (lane == 0) base = atomicAdd(stray_count, (unsigned)__popc(sm));
      base = __shfl_sync(0xffffffffu, base, 0);
      if (stray) stray_list[base + __popc(sm & ((1u << lane) - 1u))] = (int32_t)t;
    }
    if (valid && elig) {
      bool out = false;
#pragma unroll
      for (int d = 0; d < 3; ++d) out |= wrap_axis<R>(x1[d], g.L[d], g.periodic[d]);
      if (out) {
        if (w != R(0)) atomicAdd(deactivated, 1ull);
        p.w[t] = R(0);
      }
      xn[t] = x1[0]; yn[t] = x1[1]; zn[t] = x1[2];
    }
  }
  flush_all();
}

// ------------------------------------------------------------------ COOP, kernel 3: the listed particles
// (changed cell since the last sort, or changed cell in y and z at once): one thread each, global
// reductions, as in the GLOBAL design.
template <class R, int ORDER>
__global__ void __launch_bounds__(128) k_deposit_list(Grid<R> g, Particles<R> p, R* __restrict__ xn, R* __restrict__ yn,
                                                      R* __restrict__ zn, const int32_t* __restrict__ list,
                                                      const unsigned int* __restrict__ count,
                                                      unsigned long long* deactivated) {
  const unsigned n = *count;
  for (unsigned e = blockIdx.x * blockDim.x + threadIdx.x; e < n; e += gridDim.x * blockDim.x) {
    const int t = list[e];
    R x0[3] = {p.x[t], p.y[t], p.z[t]};
    R x1[3] = {xn[t], yn[t], zn[t]};
    R w = p.w[t];
    deposit_global<R, ORDER>(g, p.jf, w, x0, x1);
    bool out = false;
#pragma unroll
    for (int d = 0; d < 3; ++d) out |= wrap_axis<R>(x1[d], g.L[d], g.periodic[d]);
    if (out) {
      if (w != R(0)) atomicAdd(deactivated, 1ull);
      p.w[t] = R(0);
    }
    xn[t] = x1[0]; yn[t] = x1[1]; zn[t] = x1[2];
  }
}

// The same per-particle deposit, one WARP per listed particle: lanes 0..2 set up one axis each (compact
// window of ORDER+2 nodes: S0, DS, running sum of DS) in shared memory, then the 32 lanes walk the
// particle's nodes with x fastest, so that one RED instruction covers runs of 4-5 contiguous elements
// instead of 32 unrelated ones (L2 reduction throughput is about 2x better for contiguous lanes).
template <class R, int ORDER, int DET>
__global__ void __launch_bounds__(128) k_deposit_list_warp(Grid<R> g, Particles<R> p, R* __restrict__ xn,
                                                           R* __restrict__ yn, R* __restrict__ zn,
                                                           const int32_t* __restrict__ list,
                                                           const unsigned int* __restrict__ count,
                                                           unsigned long long* deactivated) {
  constexpr int NW = ORDER + 2;
  __shared__ R s_ax[4][3][3][NW];   // [warp][axis][S0 | DS | prefix of DS][slot]
  __shared__ int s_b[4][3];
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  const unsigned n = *count;
  const unsigned nwarps = gridDim.x * (blockDim.x >> 5);
  const R half = R(0.5), third = R(1) / R(3);
  for (unsigned e = blockIdx.x * (blockDim.x >> 5) + warp; e < n; e += nwarps) {
    const int t = list[e];
    const R w = p.w[t];
    if (lane < 3) {
      const R* a0 = lane == 0 ? p.x : (lane == 1 ? p.y : p.z);
      const R* a1 = lane == 0 ? xn : (lane == 1 ? yn : zn);
      R S0[NW], DS[NW];
      int b = esirkepov_axis<R, ORDER>(mul_rn(a0[t], g.inv_dx[lane]), mul_rn(a1[t], g.inv_dx[lane]), S0, DS);
      b = min(max(b, -kGuard), g.N[lane] + kGuard - NW);
      s_b[warp][lane] = b;
      R pre = 0;
#pragma unroll
      for (int i = 0; i < NW; ++i) {
        pre += DS[i];
        s_ax[warp][lane][0][i] = S0[i];
        s_ax[warp][lane][1][i] = DS[i];
        s_ax[warp][lane][2][i] = pre;
      }
    }
    __syncwarp();
    const int base = g.idx(s_b[warp][0], s_b[warp][1], s_b[warp][2]);
    // component d: prefix along axis d (NW-1 slots), full windows along the other two (a, b)
#pragma unroll
    for (int d = 0; d < 3; ++d) {
      const int a = d == 0 ? 1 : 0, b = d == 2 ? 1 : 2;          // the other two axes, a < b
      const R f = -(w * p.jf[d]);
      const int n0 = d == 0 ? NW - 1 : NW, n1 = d == 1 ? NW - 1 : NW, n2 = d == 2 ? NW - 1 : NW;
      for (int q = lane; q < n0 * n1 * n2; q += 32) {
        const int i = q % n0, j = (q / n0) % n1, k = q / (n0 * n1);
        const int sl[3] = {i, j, k};
        const R S0a = s_ax[warp][a][0][sl[a]], DSa = s_ax[warp][a][1][sl[a]];
        const R S0b = s_ax[warp][b][0][sl[b]], DSb = s_ax[warp][b][1][sl[b]];
        const R c = S0a * S0b + half * DSa * S0b + half * S0a * DSb + third * DSa * DSb;
        const R v = f * (s_ax[warp][d][2][sl[d]] * c);
        if (v != R(0)) j_add<R, DET>(g, g.J[d] + base + i + g.sy * j + g.sz * k, v);
      }
    }
    if (lane == 0) {
      R x1[3] = {xn[t], yn[t], zn[t]};
      bool out = false;
#pragma unroll
      for (int dd = 0; dd < 3; ++dd) out |= wrap_axis<R>(x1[dd], g.L[dd], g.periodic[dd]);
      if (out) {
        if (w != R(0)) atomicAdd(deactivated, 1ull);
        p.w[t] = R(0);
      }
      xn[t] = x1[0]; yn[t] = x1[1]; zn[t] = x1[2];
    }
    __syncwarp();
  }
}

template <class R, int ORDER>
bool launch_order(const Grid<R>& g, const ParticleStep<R>& a, int mode, Ctx& c) {
  const Particles<R>& p = a.cur;
  if (p.n == 0) return false;
  if (mode == kDepositGlobal) {
    ScopedPhase ph(c, kPhasePush);
    int64_t nb = (p.n + 127) / 128;
    k_particles_global<R, ORDER><<<(unsigned)nb, 128, 0, c.stream>>>(g, p, a.deactivated);
    c.launches++;
    return false;
  }
  R *xn = a.alt.x, *yn = a.alt.y, *zn = a.alt.z;
  cudaMemsetAsync(a.stray_count, 0, sizeof(unsigned int), c.stream);
  if (mode == kDepositTile || mode == kDepositTileMma || mode == kDepositFused) {
    // tile kernels, then the particles they listed, one warp each
    launch_tile_kernels<R>(g, a, ORDER, mode, c);
    ScopedPhase ph(c, kPhaseStray);
    auto klist = g.fix_scale[0] != 0.0 ? k_deposit_list_warp<R, ORDER, 1> : k_deposit_list_warp<R, ORDER, 0>;
    // one warp per listed particle, grid-stride; the list length is only known on the device, so the grid is sized
    // from the species: enough warps in flight for a large one (each listed particle is a chain of dependent
    // loads), few CTAs for a small one (an empty CTA still costs its launch)
    const int64_t want = p.n / 1024;
    const int blocks = (int)std::min<int64_t>((int64_t)c.sm_count * 64, std::max<int64_t>(c.sm_count, want));
    klist<<<blocks, 128, 0, c.stream>>>(g, p, xn, yn, zn, a.stray_list, a.stray_count, a.deactivated);
    c.launches += 1;
    return true;
  }
  {
    ScopedPhase ph(c, kPhasePush);
    k_push<R, ORDER><<<(unsigned)((p.n + 127) / 128), 128, 0, c.stream>>>(g, p, xn, yn, zn);
  }
  const size_t smem = (size_t)kCoopWarps * 32 * Win<ORDER>::REC * sizeof(R);
  if (c.smem_opted.insert((const void*)k_deposit_coop<R, ORDER>).second)
    cudaFuncSetAttribute(k_deposit_coop<R, ORDER>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
  const int64_t per_cta = (int64_t)kCoopWarps * kCoopChunk;
  {
    ScopedPhase ph(c, kPhaseDeposit);
    k_deposit_coop<R, ORDER><<<(unsigned)((p.n + per_cta - 1) / per_cta), kCoopWarps * 32, smem, c.stream>>>(
        g, p, xn, yn, zn, a.cell_sorted, a.stray_list, a.stray_count, a.deactivated);
  }
  {
    ScopedPhase ph(c, kPhaseStray);
    k_deposit_list<R, ORDER><<<c.sm_count * 4, 128, 0, c.stream>>>(g, p, xn, yn, zn, a.stray_list, a.stray_count,
                                                                   a.deactivated);
  }
  c.launches += 3;
  return true;
}

}  // namespace

template <class R>
bool launch_particles(const Grid<R>& g, const ParticleStep<R>& a, int order, int mode, Ctx& c) {
  switch (order) {
    case 1: return launch_order<R, 1>(g, a, mode, c);
    case 2: return launch_order<R, 2>(g, a, mode, c);
    default: return launch_order<R, 3>(g, a, mode, c);
  }
}

template bool launch_particles<double>(const Grid<double>&, const ParticleStep<double>&, int, int, Ctx&);
template bool launch_particles<float>(const Grid<float>&, const ParticleStep<float>&, int, int, Ctx&);

}  // namespace pic
