// Tile-centric particle kernels: one CTA per particle tile (<= 8x8x8 cells,
// the bins of the sort). After a sort the particles of a tile are one contiguous
// range [tile_start[t], tile_start[t+1]) in cell order, which gives the kernels their locality:
//   k_push_tile         stages the tile's E/B stencil box in shared memory once — one TMA bulk tensor copy
//                       (cp.async.bulk.tensor + mbarrier) or element-wise cp.async — then gathers and
//                       pushes one particle per thread from it (gather + push fused, no
//                       per-particle E/B in memory);
//   k_deposit_mma       Esirkepov deposition (ref [8]) as 8 x 16 x K contractions on the
//                       fp64 tensor pipe, one warp per round of 32 particles grouped by cell triple
//                       (the fp64 default);
//   k_deposit_tile      the same sums by groups of 16 lanes (4 at order 1): the lanes of a group own the
//                       (j,k) columns of a cell's window, x runs along registers (slot = node mod NX, so
//                       nothing moves when the window advances), every finished window node is one
//                       reduction at L2 (the fp32 default at orders 2 and 3);
//   k_deposit_smem_cic  fp32 order 1: lane = particle, segmented warp reduction per cell run, the tile's J
//                       box in shared memory, one flush per tile (the fp32 default at order 1);
//   k_fused_mma         gather + push + tensor-pipe deposit in one kernel (measured slower, on request).
// A particle that crosses one cell face in y or z stays in the deposit kernels (its one extra node is
// added by the warp, extra_node_deposit); particles that cross in y and z at once, or drifted too far
// from the tile since the last sort, go to a list and are deposited one warp each (particles.cu);
// correctness never depends on the order or the tile.
#include <algorithm>
#include <climits>
#include <type_traits>

#include "internal.h"
#include "particle_math.cuh"

namespace pic {

namespace {

constexpr int kTileMax = 8;   // largest tile edge (cells) these kernels are laid out for

__device__ __forceinline__ void prefetch_l2(const void* ptr) { asm volatile("prefetch.global.L2 [%0];" ::"l"(ptr)); }

// one element global -> shared without passing through registers (cp.async, 4 or 8 bytes)
template <class R>
__device__ __forceinline__ void cp_async(R* smem_dst, const R* gmem_src) {
  const unsigned sa = (unsigned)__cvta_generic_to_shared(smem_dst);
  if constexpr (sizeof(R) == 8) asm volatile("cp.async.ca.shared.global [%0], [%1], 8;" ::"r"(sa), "l"(gmem_src) : "memory");
  else asm volatile("cp.async.ca.shared.global [%0], [%1], 4;" ::"r"(sa), "l"(gmem_src) : "memory");
}

__device__ __forceinline__ void tile_coords(const TileSpec& ts, int tile, int* tb) {
  int tx = tile % ts.nt[0];
  int r = tile / ts.nt[0];
  int ty = r % ts.nt[1];
  int tz = r / ts.nt[1];
  tb[0] = tx * ts.T[0];
  tb[1] = ty * ts.T[1];
  tb[2] = tz * ts.T[2];
}

// =================================================================== gather + push from shared memory
// Box of nodes staged per component: local index 0 is node (tile base - HB); EXT nodes per axis cover
// the stencils (nodal and staggered) of every particle whose cell is inside the tile. Two layouts:
//  * TMA = false (element-wise cp.async): y fastest, then z (stride EXT), x slowest with stride SX = the
//    first value >= EXT^2 that is 9 mod 16. The lanes of a warp hold particles of a few cells that are
//    neighbours along x, so their stencil addresses differ by small multiples of SX (+-1 or +-EXT for a
//    staggered base): with SX = 9 mod 16 no two of those fall in the same pair of banks (2.10 wavefronts
//    per 64-bit load at 8 particles per cell, 2.0 is the floor), and SX odd keeps the staging stores of an
//    x-row conflict-free.
//  * TMA = true (one cp.async.bulk.tensor per CTA): the copy engine writes the box densely with the
//    array's fastest axis first, so x is fastest here; the bank spread comes from the box extents
//    instead: BX x BY x EXT nodes with BX = EXT rounded up to even (the 16-byte rule of the inner box
//    extent) and BY chosen so that the strides (1, BX, BX*BY) send the same lane patterns to distinct
//    bank pairs — 12 x 14 x 12 at order 3 gives 2.06 wavefronts per load (12 x 12 x 12 would give 3.04);
//    the BY - EXT extra rows are loaded and never read.
template <int ORDER, bool TMA = false, int ES = 8>   // ES = bytes per element
struct PushBox {
  static constexpr int HB = ORDER == 3 ? 2 : 1;
  static constexpr int EXT = kTileMax + (ORDER == 1 ? 2 : (ORDER == 2 ? 3 : 4));   // 10, 11, 12
  static constexpr int SX = EXT * EXT + ((9 - EXT * EXT % 16) + 16) % 16;            // 105, 121, 153
  // TMA: the copy must start at a 16-byte aligned address, i.e. at an x index of the padded array that is a
  // multiple of 16 / ES: with tiles that are such a multiple the box starts HBX = 16 / ES nodes below the
  // tile at every order (XOFF unused x columns where the stencils reach less far down) — a start that is
  // not aligned raises "illegal instruction" at run time. BX: >= EXT + XOFF, a multiple of 16 / ES.
  // BY from the bank simulation (fp64: 16 bank pairs, half a warp per wavefront; fp32: 32 banks, a warp).
  static constexpr int HBX = 16 / ES;                                                // 2 (fp64), 4 (fp32)
  static constexpr int XOFF = TMA ? HBX - HB : 0;                                    // local x of node (tile base - HB)
  static constexpr int BX = ES == 8 ? 12 : 16;
  static constexpr int BY = ES == 8 ? (ORDER == 1 ? 10 : 14) : (ORDER == 3 ? 13 : 11);
  static constexpr int SA = TMA ? 1 : SX;         // strides (elements) of a step along x, y, z
  static constexpr int SB = TMA ? BX : 1;
  static constexpr int SC = TMA ? BX * BY : EXT;
  static constexpr int VOL = TMA ? BX * BY * EXT : EXT * SX;
  static constexpr int MAXD = 256;   // drifted particles a CTA lists before it gathers them in line
};

// NX, NY, NZ weights per axis: ORDER + 1, or ORDER along a staggered axis of the Galerkin gather
template <class R, int ORDER, bool TMA, int NX = ORDER + 1, int NY = ORDER + 1, int NZ = ORDER + 1>
__device__ __forceinline__ R interp_box(const R* __restrict__ F, int base, const R* wx, const R* wy, const R* wz) {
  using PB = PushBox<ORDER, TMA, (int)sizeof(R)>;
  constexpr int SA = PB::SA, SB = PB::SB, SC = PB::SC;
  R acc = 0;
  if constexpr (kStatementOrder<R>) {   // sum over c, b, a (a innermost) of ((wx wy) wz) F, every operation rounded
#pragma unroll
    for (int c = 0; c < NZ; ++c)
#pragma unroll
      for (int b = 0; b < NY; ++b)
#pragma unroll
        for (int a = 0; a < NX; ++a)
          acc = add_rn(acc, mul_rn(mul_rn(mul_rn(wx[a], wy[b]), wz[c]), F[base + SA * a + SB * b + SC * c]));
  } else {
#pragma unroll
    for (int c = 0; c < NZ; ++c) {
      R accb = 0;
#pragma unroll
      for (int b = 0; b < NY; ++b) {
        R acca = 0;
#pragma unroll
        for (int a = 0; a < NX; ++a) acca += wx[a] * F[base + SA * a + SB * b + SC * c];
        accb += wy[b] * acca;
      }
      acc += wz[c] * accb;
    }
  }
  return acc;
}

// ---- TMA + mbarrier primitives (sm_90+ PTX; SASS: UTMALDG, SYNCS)
__device__ __forceinline__ void mbar_init(unsigned long long* bar, unsigned count) {
  asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"((unsigned)__cvta_generic_to_shared(bar)), "r"(count) : "memory");
}
__device__ __forceinline__ void mbar_expect_tx(unsigned long long* bar, unsigned bytes) {
  asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"((unsigned)__cvta_generic_to_shared(bar)), "r"(bytes)
               : "memory");
}
__device__ __forceinline__ void mbar_wait(unsigned long long* bar, unsigned parity) {
  const unsigned a = (unsigned)__cvta_generic_to_shared(bar);
  asm volatile(
      "{\n"
      ".reg .pred p;\n"
      "WAIT_%=:\n"
      "mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n"
      "@p bra DONE_%=;\n"
      "bra WAIT_%=;\n"
      "DONE_%=:\n"
      "}" ::"r"(a), "r"(parity)
      : "memory");
}
// one 4-D tile (x, y, z, component) of the tensor `tmap` describes -> shared memory, completion on `bar`;
// coordinates may start below 0 or end past the tensor: those elements arrive as zeros
__device__ __forceinline__ void tma_load_4d(void* smem_dst, const CUtensorMap* tmap, unsigned long long* bar, int c0, int c1,
                                            int c2, int c3) {
  asm volatile(
      "cp.async.bulk.tensor.4d.shared::cluster.global.tile.mbarrier::complete_tx::bytes [%0], [%1, {%3, %4, %5, %6}], [%2];" ::"r"(
          (unsigned)__cvta_generic_to_shared(smem_dst)),
      "l"(tmap), "r"((unsigned)__cvta_generic_to_shared(bar)), "r"(c0), "r"(c1), "r"(c2), "r"(c3)
      : "memory");
}

template <class R, int PUSHER>
__device__ __forceinline__ void push_store(const Grid<R>& g, const Particles<R>& p, R* __restrict__ xn,
                                           R* __restrict__ yn, R* __restrict__ zn, int t, const R* x0, R* u,
                                           const R* Ef, const R* Bf) {
  push_momentum<R>(PUSHER, p.kq, g.inv_c2, Ef, Bf, u);   // compile-time constant: the other branch folds away
  R x1[3];
  advance<R>(g.dt, g.inv_c2, x0, u, x1);
  xn[t] = x1[0]; yn[t] = x1[1]; zn[t] = x1[2];
  p.ux[t] = u[0]; p.uy[t] = u[1]; p.uz[t] = u[2];
}

// Pusher (PIC_PUSHER_*) and gather variant (PIC_GATHER_*) are template parameters: four instantiations
// per order and precision, (0, 0) being the default and benchmarked path. The Galerkin gather carries one
// weight less along every staggered axis, so it reads 288 box elements per particle instead of 384 at
// order 3 — and runs faster by that ratio, since those reads are what bounds the kernel.
// TMA: the box arrives by ONE bulk tensor copy issued by one thread (all six components: the field arrays
// are one allocation, described as a 4-D tensor), signalled on an mbarrier; meanwhile every thread already
// loads its first particle. Otherwise 6 * EXT^3 element-wise cp.async copies.
template <class R, int ORDER, int PUSHER, int GATHER, bool TMA>
// Register budget: two CTAs per SM (128 registers) where the box needs the shared memory anyway; fp32 at order
// 1 (25 KB box) is latency-bound instead and runs best with four (64 registers; C3 push by CTAs per SM:
// 2: 0.395 ms, 3: 0.333, 4: 0.316, 5: 0.318, 6: 0.334)
__global__ void __launch_bounds__(kPushTileThreads<R>, (sizeof(R) == 4 && ORDER == 1) ? 4 : 2) k_push_tile(Grid<R> g, Particles<R> p, R* __restrict__ xn,
                                                                   R* __restrict__ yn, R* __restrict__ zn,
                                                                   const int32_t* __restrict__ tile_start, TileSpec ts,
                                                                   const __grid_constant__ CUtensorMap tmap) {
  using PB = PushBox<ORDER, TMA, (int)sizeof(R)>;
  constexpr int E = PB::EXT, VOL = PB::VOL, SA = PB::SA, SB = PB::SB, SC = PB::SC;
  constexpr int NS = GATHER == 1 ? ORDER : ORDER + 1;   // weights along a staggered axis
  constexpr int NN = ORDER + 1;
  extern __shared__ __align__(128) unsigned char smem_raw[];
  R* box_raw = reinterpret_cast<R*>(smem_raw);   // [6][VOL]
  R* box = box_raw + PB::XOFF * SA;              // local (0,0,0) = node (tile base - HB)
  __shared__ int s_drift[PB::MAXD];
  __shared__ int s_ndrift;
  __shared__ __align__(8) unsigned long long s_bar;
  const int tile = blockIdx.x;
  const int s = tile_start[tile], e = tile_start[tile + 1];
  if (s >= e) return;
  if (threadIdx.x == 0) s_ndrift = 0;
  int tb[3];
  tile_coords(ts, tile, tb);
  const int o0 = tb[0] - PB::HB, o1 = tb[1] - PB::HB, o2 = tb[2] - PB::HB;   // node of local (0,0,0)
  if constexpr (TMA) {
    if (threadIdx.x == 0) {
      mbar_init(&s_bar, 1);
      asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
      mbar_expect_tx(&s_bar, (unsigned)(6 * VOL * sizeof(R)));
      tma_load_4d(box_raw, &tmap, &s_bar, tb[0] - PB::HBX + kGuard, o1 + kGuard, o2 + kGuard, 0);
    }
    __syncthreads();   // the barrier object (and s_ndrift) visible to every thread before anyone waits on it
  } else {
    // stage the six boxes, reading along x (nodes beyond the padded array, possible only for tiles
    // smaller than 8, read 0)
    const int lim0 = g.N[0] + kGuard, lim1 = g.N[1] + kGuard, lim2 = g.N[2] + kGuard;
    for (int idx = threadIdx.x; idx < E * E * E; idx += blockDim.x) {
      int i = idx % E, r = idx / E;
      int j = r % E, k = r / E;
      const bool in = (o0 + i < lim0) & (o1 + j < lim1) & (o2 + k < lim2);
      const int gi = g.idx(o0 + i, o1 + j, o2 + k);
      const int li = SA * i + SB * j + SC * k;
      // asynchronous copies (LDGSTS): every element of the box is in flight at once, no register staging
#pragma unroll
      for (int c = 0; c < 6; ++c) {
        if (in) cp_async(box + c * VOL + li, g.F[c] + gi);
        else box[c * VOL + li] = R(0);
      }
    }
  }
  bool staged = !TMA;
  if constexpr (!TMA) {
    asm volatile("cp.async.wait_all;" ::: "memory");
    __syncthreads();
  }
  for (int t = s + threadIdx.x; t < e; t += blockDim.x) {
    R x0[3] = {p.x[t], p.y[t], p.z[t]};
    R u[3] = {p.ux[t], p.uy[t], p.uz[t]};
    if (t + (int)blockDim.x < e) {   // the next particle of this thread on its way to L2
      const int tn = t + blockDim.x;
      prefetch_l2(p.x + tn); prefetch_l2(p.y + tn); prefetch_l2(p.z + tn);
      prefetch_l2(p.ux + tn); prefetch_l2(p.uy + tn); prefetch_l2(p.uz + tn);
    }
    R wn[3][ORDER + 1], ws[3][ORDER + 1];
    int ln[3], ls[3];
    bool inbox = true;
#pragma unroll
    for (int d = 0; d < 3; ++d) {
      const R xi = mul_rn(x0[d], g.inv_dx[d]);
      const R xs = sub_rn(xi, R(0.5));
      ln[d] = shape<R, ORDER>(xi, wn[d]) - (d == 0 ? o0 : (d == 1 ? o1 : o2));
      ls[d] = (GATHER == 1 ? shape_lowered<R, ORDER>(xs, ws[d]) : shape<R, ORDER>(xs, ws[d])) -
              (d == 0 ? o0 : (d == 1 ? o1 : o2));
      inbox &= (ln[d] >= 0) & (ln[d] <= E - ORDER - 1) & (ls[d] >= 0) & (ls[d] <= E - ORDER - 1);
    }
    if constexpr (TMA) {
      if (!staged) {   // the box has been on its way while the first particle was loaded and its weights formed
        mbar_wait(&s_bar, 0);
        staged = true;
      }
    }
    if (!inbox) {
      // drifted out of the tile since the last sort: listed, gathered from global memory below with all
      // lanes busy. If the list overflows the entry is dropped and the second pass finds these particles by
      // walking the tile again: ONE copy of the global-memory gather, so that a particle's result never
      // depends on which threads reached the list first (bit-identical runs, pic_options.deterministic)
      const int slot = atomicAdd(&s_ndrift, 1);
      if (slot < PB::MAXD) s_drift[slot] = t;
      continue;
    }
    R Ef[3], Bf[3];
    // Ex (s,n,n)  Ey (n,s,n)  Ez (n,n,s)  Bx (n,s,s)  By (s,n,s)  Bz (s,s,n)
    Ef[0] = interp_box<R, ORDER, TMA, NS, NN, NN>(box + 0 * VOL, SA * ls[0] + SB * ln[1] + SC * ln[2], ws[0], wn[1], wn[2]);
    Ef[1] = interp_box<R, ORDER, TMA, NN, NS, NN>(box + 1 * VOL, SA * ln[0] + SB * ls[1] + SC * ln[2], wn[0], ws[1], wn[2]);
    Ef[2] = interp_box<R, ORDER, TMA, NN, NN, NS>(box + 2 * VOL, SA * ln[0] + SB * ln[1] + SC * ls[2], wn[0], wn[1], ws[2]);
    Bf[0] = interp_box<R, ORDER, TMA, NN, NS, NS>(box + 3 * VOL, SA * ln[0] + SB * ls[1] + SC * ls[2], wn[0], ws[1], ws[2]);
    Bf[1] = interp_box<R, ORDER, TMA, NS, NN, NS>(box + 4 * VOL, SA * ls[0] + SB * ln[1] + SC * ls[2], ws[0], wn[1], ws[2]);
    Bf[2] = interp_box<R, ORDER, TMA, NS, NS, NN>(box + 5 * VOL, SA * ls[0] + SB * ls[1] + SC * ln[2], ws[0], ws[1], wn[2]);
    push_store<R, PUSHER>(g, p, xn, yn, zn, t, x0, u, Ef, Bf);
  }
  __syncthreads();
  const int nd = s_ndrift;
  const bool rescan = nd > PB::MAXD;   // warp-uniform (CTA-uniform)
  const int cnt = rescan ? e - s : nd;
  for (int q = threadIdx.x; q < cnt; q += blockDim.x) {
    const int t = rescan ? s + q : s_drift[q];
    R x0[3] = {p.x[t], p.y[t], p.z[t]};
    if (rescan) {   // the same test as above, on the same bits
      bool inbox = true;
#pragma unroll
      for (int d = 0; d < 3; ++d) {
        R wtmp[ORDER + 1];
        const R xi = mul_rn(x0[d], g.inv_dx[d]);
        const R xs = sub_rn(xi, R(0.5));
        const int od = d == 0 ? o0 : (d == 1 ? o1 : o2);
        const int l_n = shape<R, ORDER>(xi, wtmp) - od;
        const int l_s = (GATHER == 1 ? shape_lowered<R, ORDER>(xs, wtmp) : shape<R, ORDER>(xs, wtmp)) - od;
        inbox &= (l_n >= 0) & (l_n <= E - ORDER - 1) & (l_s >= 0) & (l_s <= E - ORDER - 1);
      }
      if (inbox) continue;
    }
    R u[3] = {p.ux[t], p.uy[t], p.uz[t]};
    R Ef[3], Bf[3];
    gather6<R, ORDER, GATHER != 0>(g, x0[0], x0[1], x0[2], Ef, Bf);
    push_store<R, PUSHER>(g, p, xn, yn, zn, t, x0, u, Ef, Bf);
  }
}

// =================================================================== Esirkepov deposition per tile
template <class R>
struct alignas(2 * sizeof(R)) Pair2 { R a, b; };

// Windows fixed to a CELL c (the cell of the old position): x nodes c-BLX .. c-BLX+NX-1 cover any
// move of up to one cell along x; y and z nodes c-BLYZ .. c-BLYZ+NYZ-1 cover the moves that stay in
// the cell along that axis (the others go to the list). NYZ^2 lanes own the (j,k) columns.
template <int ORDER>
struct TWin {
  static constexpr int NX = ORDER == 1 ? 4 : 6, BLX = ORDER == 1 ? 1 : 2;
  static constexpr int NYZ = ORDER == 1 ? 2 : 4, BLYZ = ORDER == 1 ? 0 : 1;
  static constexpr int LG = NYZ * NYZ;                 // lanes per particle: 4 or 16
  // record (elements): {A_x,B_x}[NX] | PX[NX] | {S0_y,DS_y}[NYZ] | PY[NYZ] | {S0_z,DS_z}[NYZ] | PZ[NYZ]
  static constexpr int oAB = 0, oPX = 2 * NX, oY = 3 * NX, oPY = 3 * NX + 2 * NYZ, oZ = 3 * NX + 3 * NYZ,
                       oPZ = 3 * NX + 5 * NYZ;
  static constexpr int RAW = 3 * NX + 6 * NYZ;                     // 42 / 24
  static constexpr int REC = (RAW / 2) % 2 == 1 ? RAW : RAW + 2;   // REC/2 odd: conflict-free pair stores
};

// old/new weights of one axis placed on an NW-node window whose first node is (cell - BL), where
// `cell` is the cell of the OLD position; `fits` = both supports lie inside the window. For orders 1
// and 3 the old support starts at a fixed slot (cell - 1 + ... is static), so only the new weights
// need selects.
template <class R, int ORDER, int NW, int BL>
__device__ __forceinline__ void axis_window_from(int l0, const R* w0, R xi0, R xi1, int& cell, R* S0, R* DS, bool& fits) {
  R w1[ORDER + 1];
  const int l1 = shape<R, ORDER>(xi1, w1);
  const int c = ORDER == 2 ? (int)floor(xi0) : (ORDER == 1 ? l0 : l0 + 1);
  cell = c;
  if constexpr (ORDER != 2 && NW == ORDER + 1) {
    // tight window: it is the old support itself; the new one fits only if it starts at the same node
#pragma unroll
    for (int i = 0; i < NW; ++i) { S0[i] = w0[i]; DS[i] = sub_rn(w1[i], w0[i]); }
    fits = l1 == l0;
    return;
  } else if constexpr (ORDER != 2 && NW == ORDER + 3) {
    // old support at slots 1..ORDER+1; the new one starts at slot 0, 1 or 2
    const int sl1 = l1 - l0 + 1;
    const bool d0 = sl1 == 0, d2 = sl1 == 2;
#pragma unroll
    for (int i = 0; i < NW; ++i) {
      const R lo = i <= ORDER ? w1[i <= ORDER ? i : 0] : R(0);
      const R mid = (i >= 1 && i <= ORDER + 1) ? w1[(i >= 1 && i <= ORDER + 1) ? i - 1 : 0] : R(0);
      const R hi = i >= 2 ? w1[i >= 2 ? i - 2 : 0] : R(0);
      const R a = (i >= 1 && i <= ORDER + 1) ? w0[(i >= 1 && i <= ORDER + 1) ? i - 1 : 0] : R(0);
      const R b = d0 ? lo : (d2 ? hi : mid);
      S0[i] = a;
      DS[i] = sub_rn(b, a);
    }
    fits = (sl1 >= 0) & (sl1 <= 2);
    return;
  }
  const int so0 = ORDER == 2 ? l0 - (c - BL) : (ORDER == 1 ? BL : BL - 1);
  const int sl1 = l1 - (c - BL);
#pragma unroll
  for (int i = 0; i < NW; ++i) {
    R a = 0, b = 0;
#pragma unroll
    for (int k = 0; k <= ORDER; ++k) {
      a = (i == so0 + k) ? w0[k] : a;
      b = (i == sl1 + k) ? w1[k] : b;
    }
    S0[i] = a;
    DS[i] = sub_rn(b, a);
  }
  fits = (so0 >= 0) & (so0 + ORDER < NW) & (sl1 >= 0) & (sl1 + ORDER < NW);
}

template <class R, int ORDER, int NW, int BL>
__device__ __forceinline__ void axis_window(R xi0, R xi1, int& cell, R* S0, R* DS, bool& fits) {
  R w0[ORDER + 1];
  const int l0 = shape<R, ORDER>(xi0, w0);
  axis_window_from<R, ORDER, NW, BL>(l0, w0, xi0, xi1, cell, S0, DS, fits);
}

// The y and z windows are tied to the old cell and hold exactly the moves that stay in it. A particle that
// crosses ONE cell face along the axis has a new support that sticks out of the window by one node, below
// (ext = 1, window slot -1) or above (ext = 2, slot NW), where its old weight is zero and its new one is
// `dext`; the NW window slots are filled as always (DS = new - old, the new weights shifted by one slot).
// Esirkepov's J is a sum over nodes that is linear in the pair (S0, DS) of every single node, so the window
// part goes through the tile kernels' contractions unchanged and the one extra node is added separately
// (extra_node_deposit below). ext = 0: fits; ext = 3: further out (per-particle pass).
template <class R, int ORDER, int NW, int BL>
__device__ __forceinline__ void axis_window_ext(R xi0, R xi1, int& cell, R* S0, R* DS, int& ext, R& dext) {
  R w0[ORDER + 1], w1[ORDER + 1];
  const int l0 = shape<R, ORDER>(xi0, w0);
  const int l1 = shape<R, ORDER>(xi1, w1);
  const int c = ORDER == 2 ? (int)floor(xi0) : (ORDER == 1 ? l0 : l0 + 1);
  cell = c;
  const int so0 = l0 - (c - BL);   // static for orders 1 and 3
  const int sl1 = l1 - (c - BL);
  if constexpr (ORDER != 2 && NW == ORDER + 1) {
    // tight window: it is the old support itself; the new one starts at slot -1, 0 or +1
    const int sh = l1 - l0;
#pragma unroll
    for (int i = 0; i < NW; ++i) {
      const R up = i >= 1 ? w1[i >= 1 ? i - 1 : 0] : R(0);          // sh = +1
      const R dn = i + 1 < NW ? w1[i + 1 < NW ? i + 1 : 0] : R(0);  // sh = -1
      const R b = sh == 0 ? w1[i] : (sh > 0 ? up : dn);
      S0[i] = w0[i];
      DS[i] = sub_rn(b, w0[i]);
    }
    ext = sh == 0 ? 0 : (sh == -1 ? 1 : (sh == 1 ? 2 : 3));
    dext = sh < 0 ? w1[0] : w1[ORDER];
  } else {
#pragma unroll
    for (int i = 0; i < NW; ++i) {
      R a = 0, b = 0;
#pragma unroll
      for (int k = 0; k <= ORDER; ++k) {
        a = (i == so0 + k) ? w0[k] : a;
        b = (i == sl1 + k) ? w1[k] : b;
      }
      S0[i] = a;
      DS[i] = sub_rn(b, a);
    }
    const bool oldfits = (so0 >= 0) & (so0 + ORDER < NW);
    const bool fits = (sl1 >= 0) & (sl1 + ORDER < NW);
    ext = !oldfits ? 3 : (fits ? 0 : (sl1 == -1 ? 1 : (sl1 + ORDER == NW ? 2 : 3)));
    dext = sl1 < 0 ? w1[0] : w1[ORDER];
  }
}

// The extra node of the particles of a round that crossed a face in y or in z (axis_window_ext): for each
// of them the warp adds the contributions of that one node, lane = (i, m) with i the NX window nodes along x
// (fastest: contiguous reductions) and m the window slots of the other transverse axis. At the extra node
// the old weight is 0 and the new one d, hence with (S0, DS) = (0, d) along the crossing axis e, o the other
// transverse axis and A = S0x + DSx/2, B = S0x/2 + DSx/3 (all in the particle's record):
//   Jx = PX[i] d (S0o[m]/2 + DSo[m]/3),   Jo = Po[m] d B[i],   Je = f_e (running sum of DS_e) (A[i] S0o[m] + B[i] DSo[m]),
// the running sum through the extra node being d below the window and the total, 0, above it.
// extc: 0 none, 1/2 y below/above, 5/6 z below/above; fext = f_e d for a node below, else 0. Warp-uniform.
// Nothing but extc is kept across the contraction: the owning lane recomputes d (same expression, same bits)
// from the new position it still holds for the store.
template <class R, int ORDER, int DET, class W>
__device__ __forceinline__ void extra_node_deposit_warp(const Grid<R>& g, const R* __restrict__ rec, unsigned em, int extc,
                                                     R x1y, R x1z, R w, const R* jf, int wx0, int wy0, int wz0) {
  constexpr int NX = W::NX, NYZ = W::NYZ;
  const int lane = threadIdx.x & 31;
  const R half = R(0.5), third = R(1) / R(3);
  R dext = 0, fext = 0;
  if (extc != 0) {
    const int e = extc < 4 ? 1 : 2;
    R w1[ORDER + 1];
    shape<R, ORDER>(mul_rn(e == 1 ? x1y : x1z, g.inv_dx[e]), w1);
    const bool below = (extc & 3) == 1;
    dext = below ? w1[0] : w1[ORDER];
    fext = below ? -(w * jf[e]) * dext : R(0);
  }
  while (em) {
    const int src = __ffs(em) - 1;
    em &= em - 1;
    const int ec = __shfl_sync(0xffffffffu, extc, src);
    const R d = __shfl_sync(0xffffffffu, dext, src);
    const R fe = __shfl_sync(0xffffffffu, fext, src);
    const int X0 = __shfl_sync(0xffffffffu, wx0, src), Y0 = __shfl_sync(0xffffffffu, wy0, src),
              Z0 = __shfl_sync(0xffffffffu, wz0, src);
    if (lane < NX * NYZ) {
      const R* rr = rec + src * W::REC;
      const int i = lane % NX, m = lane / NX;
      const bool isy = ec < 4;
      const int eo = (ec & 3) == 1 ? -1 : NYZ;
      const Pair2<R> ab = *reinterpret_cast<const Pair2<R>*>(rr + W::oAB + 2 * i);
      const R px = rr[W::oPX + i];
      const Pair2<R> ov = *reinterpret_cast<const Pair2<R>*>(rr + (isy ? W::oZ : W::oY) + 2 * m);
      const R po = rr[(isy ? W::oPZ : W::oPY) + m];
      const R vx = px * (d * (half * ov.a + third * ov.b));
      const R vo = po * (d * ab.b);
      const R ve = fe * (ab.a * ov.a + ab.b * ov.b);
      const int base = g.idx(X0 + i, isy ? Y0 + eo : Y0 + m, isy ? Z0 + m : Z0 + eo);
      if (vx != R(0)) j_add<R, DET>(g, g.J[0] + base, vx);
      if (vo != R(0)) j_add<R, DET>(g, g.J[isy ? 2 : 1] + base, vo);
      if (ve != R(0)) j_add<R, DET>(g, g.J[isy ? 1 : 2] + base, ve);
    }
  }
}

template <class R, int ORDER, int DET, class W>
__device__ __forceinline__ void extra_node_deposit(const Grid<R>& g, const R* __restrict__ rec, int extc, R x1y, R x1z,
                                                   R w, const R* jf, int wx0, int wy0, int wz0) {
  const unsigned em = __ballot_sync(0xffffffffu, extc != 0);
  if (em != 0) extra_node_deposit_warp<R, ORDER, DET, W>(g, rec, em, extc, x1y, x1z, w, jf, wx0, wy0, wz0);
}


// One particle's record (layout W: {A_x,B_x}[NX] | PX[NX] | {S0_y,DS_y}[NYZ] | PY[NYZ] | {S0_z,DS_z}[NYZ] | PZ[NYZ]),
// written axis by axis as soon as the axis is known, so that only one axis' weights are live at a time
// (a record whose particle turns out not to fit is simply never read). Returns the cell of the old
// position in c[], whether the move fits the windows (x: +-1 cell; y, z: same cell, or ONE face of ONE
// of the two crossed) and in `extc` the extra node of such a crossing (extra_node_deposit).
template <class R, int ORDER, class W>
__device__ __forceinline__ bool build_record(const Grid<R>& g, const R* jf, R* __restrict__ rr, const R* x0,
                                             const R* x1, R w, int* c, int& extc) {
  constexpr int NX = W::NX, NYZ = W::NYZ;
  const R half = R(0.5), third = R(1) / R(3);
  bool fitx;
  {
    R S0[NX], DS[NX];
    axis_window<R, ORDER, NX, W::BLX>(mul_rn(x0[0], g.inv_dx[0]), mul_rn(x1[0], g.inv_dx[0]), c[0], S0, DS, fitx);
    const R fx = -(w * jf[0]);
    R px = 0;
#pragma unroll
    for (int i = 0; i < NX; ++i) {
      *reinterpret_cast<Pair2<R>*>(rr + W::oAB + 2 * i) = Pair2<R>{S0[i] + half * DS[i], half * S0[i] + third * DS[i]};
      px += DS[i];
      rr[W::oPX + i] = fx * px;
    }
  }
  int e[2];
#pragma unroll
  for (int a = 0; a < 2; ++a) {   // y, z
    R S0[NYZ], DS[NYZ], d;
    axis_window_ext<R, ORDER, NYZ, W::BLYZ>(mul_rn(x0[1 + a], g.inv_dx[1 + a]), mul_rn(x1[1 + a], g.inv_dx[1 + a]),
                                            c[1 + a], S0, DS, e[a], d);
    const R f = -(w * jf[1 + a]);
    R pr = e[a] == 1 ? d : R(0);   // running sum of DS: a node below the window comes first
    const int oS = a == 0 ? W::oY : W::oZ, oP = a == 0 ? W::oPY : W::oPZ;
#pragma unroll
    for (int i = 0; i < NYZ; ++i) {
      *reinterpret_cast<Pair2<R>*>(rr + oS + 2 * i) = Pair2<R>{S0[i], DS[i]};
      pr += DS[i];
      rr[oP + i] = f * pr;
    }
  }
  extc = e[0] ? e[0] : (e[1] ? 4 + e[1] : 0);
  return fitx & (e[0] < 3) & (e[1] < 3) & ((e[0] == 0) | (e[1] == 0));
}

// Register accumulators of one lane: the (j,k) column of a window of NX nodes along x, three
// components. The slot of box node X is X mod NX, so when the window advances by one cell nothing
// moves: the slot of the node that left is flushed and reused for the node that entered.
template <class R, int NX>
struct Acc {
  R x[NX], y[NX], z[NX];
  __device__ __forceinline__ void zero() {
#pragma unroll
    for (int i = 0; i < NX; ++i) { x[i] = 0; y[i] = 0; z[i] = 0; }
  }
};

// one particle's contribution to this lane's column; PH = (first box node of the window) mod NX
template <class R, int ORDER, int PH>
__device__ __forceinline__ void accumulate(Acc<R, TWin<ORDER>::NX>& a, const R* __restrict__ rr, int j, int k) {
  using W = TWin<ORDER>;
  constexpr int NX = W::NX;
  const R half = R(0.5), third = R(1) / R(3);
  const Pair2<R> yv = *reinterpret_cast<const Pair2<R>*>(rr + W::oY + 2 * j);
  const Pair2<R> zv = *reinterpret_cast<const Pair2<R>*>(rr + W::oZ + 2 * k);
  const R py = rr[W::oPY + j], pz = rr[W::oPZ + k];
  const R cx = zv.a * (yv.a + half * yv.b) + zv.b * (half * yv.a + third * yv.b);
  const R q1 = py * zv.a, q2 = py * zv.b;
  const R r1 = pz * yv.a, r2 = pz * yv.b;
#pragma unroll
  for (int i = 0; i < NX; ++i) {
    const int P = (PH + i) % NX;   // static after unrolling
    const Pair2<R> ab = *reinterpret_cast<const Pair2<R>*>(rr + W::oAB + 2 * i);
    if (i < NX - 1) a.x[P] = fma(cx, rr[W::oPX + i], a.x[P]);
    a.y[P] = fma(q1, ab.a, fma(q2, ab.b, a.y[P]));
    a.z[P] = fma(r1, ab.a, fma(r2, ab.b, a.z[P]));
  }
}

// where a window's first node lives in the three J arrays
template <class R>
struct JPtr { R* p[3]; };

// sum over the NG groups of a warp (lanes that own the same column), result in every lane
template <class R, int LG>
__device__ __forceinline__ R group_sum(R v) {
#pragma unroll
  for (int o = LG; o < 32; o <<= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
  return v;
}

// one physical slot (static P), summed over the groups -> the J element jx points at, then cleared.
// Warp-uniform.
template <class R, int ORDER, int P, int DET>
__device__ __forceinline__ void flush_slot(const Grid<R>& g, Acc<R, TWin<ORDER>::NX>& a, const JPtr<R>& jx, bool writer) {
  using W = TWin<ORDER>;
  const R vx = group_sum<R, W::LG>(a.x[P]), vy = group_sum<R, W::LG>(a.y[P]), vz = group_sum<R, W::LG>(a.z[P]);
  if (writer) {
    if (vx != R(0)) j_add<R, DET>(g, jx.p[0], vx);
    if (vy != R(0)) j_add<R, DET>(g, jx.p[1], vy);
    if (vz != R(0)) j_add<R, DET>(g, jx.p[2], vz);
  }
  a.x[P] = 0; a.y[P] = 0; a.z[P] = 0;
}

// all slots: physical slot p holds logical slot (p - ph) mod NX of the window at jx. Warp-uniform.
template <class R, int ORDER, int DET>
__device__ __forceinline__ void flush_window(const Grid<R>& g, Acc<R, TWin<ORDER>::NX>& a, const JPtr<R>& jx, int ph, bool writer) {
  using W = TWin<ORDER>;
  constexpr int NX = W::NX;
#pragma unroll
  for (int p = 0; p < NX; ++p) {
    int i = p - ph;
    i += i < 0 ? NX : 0;
    const R vx = group_sum<R, W::LG>(a.x[p]), vy = group_sum<R, W::LG>(a.y[p]), vz = group_sum<R, W::LG>(a.z[p]);
    if (writer) {
      if (vx != R(0)) j_add<R, DET>(g, jx.p[0] + i, vx);
      if (vy != R(0)) j_add<R, DET>(g, jx.p[1] + i, vy);
      if (vz != R(0)) j_add<R, DET>(g, jx.p[2] + i, vz);
    }
  }
  a.zero();
}

// the particles of one cell (cnt of them, record slots listed in order[]): NG at a time, one per
// group. PH = (first box node of the cell's window) mod NX; adv = the window moved up one cell.
template <class R, int ORDER, int PH, int DET>
__device__ __forceinline__ void cell_batch(const Grid<R>& g, Acc<R, TWin<ORDER>::NX>& a, bool adv, const JPtr<R>& jx_old, bool writer,
                                           const R* __restrict__ rec, const int* __restrict__ order, int cnt, int grp,
                                           int j, int k) {
  using W = TWin<ORDER>;
  constexpr int NX = W::NX, NG = 32 / W::LG;
  if (adv) flush_slot<R, ORDER, (PH + NX - 1) % NX, DET>(g, a, jx_old, writer);
#pragma unroll 1
  for (int it = grp; it < cnt; it += NG) accumulate<R, ORDER, PH>(a, rec + order[it] * W::REC, j, k);
}

// Every finished window node is one reduction at L2 (RED.ADD.F64 / .F32): no J box in shared memory,
// no prologue / epilogue, no block barrier, so two 8-warp CTAs per SM overlap freely.
template <class R, int ORDER, int NWARP, int DET>
__global__ void __launch_bounds__(NWARP * 32, 2)
    k_deposit_tile(Grid<R> g, Particles<R> p, R* __restrict__ xn, R* __restrict__ yn, R* __restrict__ zn,
                   const int32_t* __restrict__ tile_start, TileSpec ts, int32_t* __restrict__ stray_list,
                   unsigned int* __restrict__ stray_count, unsigned long long* deactivated) {
  using W = TWin<ORDER>;
  constexpr int NX = W::NX, NYZ = W::NYZ, LG = W::LG, REC = W::REC;
  constexpr bool kExt = ORDER != 1;   // extra node of a face crossing in y or z taken here (see below)
  extern __shared__ __align__(128) unsigned char smem_raw[];
  R* rec_all = reinterpret_cast<R*>(smem_raw);
  __shared__ int s_order[NWARP][32];

  const int tile = blockIdx.x;
  const int s = tile_start[tile], e = tile_start[tile + 1];
  if (s >= e) return;
  int tb[3];
  tile_coords(ts, tile, tb);

  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  const int grp = lane / LG, gl = lane % LG;
  const int j = gl % NYZ, k = gl / NYZ;
  // first node of this lane's (j,k) column of the window whose box offset is `off`
  const int b0 = tb[0] - W::BLX, b1 = tb[1] - W::BLYZ, b2 = tb[2] - W::BLYZ;
  auto column = [&](int off) {
    JPtr<R> q;
    const int gi = g.idx(b0 + (off & 15), b1 + ((off >> 4) & 15) + j, b2 + (off >> 8) + k);
    q.p[0] = g.J[0] + gi; q.p[1] = g.J[1] + gi; q.p[2] = g.J[2] + gi;
    return q;
  };
  R* rec = rec_all + (size_t)warp * 32 * REC;
  const R half = R(0.5), third = R(1) / R(3);

  // the warp's contiguous share of the tile, a multiple of 32 particles
  const int n = e - s;
  const int chunk = ((n + NWARP - 1) / NWARP + 31) & ~31;
  const int wb = s + warp * chunk;
  const int we = min(e, wb + chunk);

  Acc<R, NX> acc;
  acc.zero();
  int cur = INT_MIN;   // box offset of the window being accumulated (its first node), per group
  int curph = 0;       // (x index of that node) mod NX

  for (int rb = wb; rb < we; rb += 32) {
    const int t = rb + lane;
    const bool valid = t < we;
    bool elig = false;
    R x1[3] = {0, 0, 0};
    R w = 0;
    int code = -1;
    int extc = 0;           // extra node of a particle that crossed a face in y or z (extra_node_deposit)
    if (valid) {
      R x0[3] = {p.x[t], p.y[t], p.z[t]};
      x1[0] = xn[t]; x1[1] = yn[t]; x1[2] = zn[t];
      w = p.w[t];
      // all three axes first, the record only if the move fits (this kernel has the registers for it; at
      // order 1 in fp32 that order of things is 20 % faster than build_record's axis-by-axis stores, and the
      // extra node is left out there: measured on C3, taking it in line costs 0.16 ms and saves 0.05 ms of the
      // per-particle pass)
      R S0x[NX], DSx[NX], S0y[NYZ], DSy[NYZ], S0z[NYZ], DSz[NYZ];
      int c[3];
      bool fitx, fityz;
      int ey = 0, ez = 0;
      R dy = 0, dz = 0;
      axis_window<R, ORDER, NX, W::BLX>(mul_rn(x0[0], g.inv_dx[0]), mul_rn(x1[0], g.inv_dx[0]), c[0], S0x, DSx, fitx);
      if constexpr (kExt) {
        axis_window_ext<R, ORDER, NYZ, W::BLYZ>(mul_rn(x0[1], g.inv_dx[1]), mul_rn(x1[1], g.inv_dx[1]), c[1], S0y, DSy, ey, dy);
        axis_window_ext<R, ORDER, NYZ, W::BLYZ>(mul_rn(x0[2], g.inv_dx[2]), mul_rn(x1[2], g.inv_dx[2]), c[2], S0z, DSz, ez, dz);
        fityz = (ey < 3) & (ez < 3) & ((ey == 0) | (ez == 0));
      } else {
        bool fy_, fz_;
        axis_window<R, ORDER, NYZ, W::BLYZ>(mul_rn(x0[1], g.inv_dx[1]), mul_rn(x1[1], g.inv_dx[1]), c[1], S0y, DSy, fy_);
        axis_window<R, ORDER, NYZ, W::BLYZ>(mul_rn(x0[2], g.inv_dx[2]), mul_rn(x1[2], g.inv_dx[2]), c[2], S0z, DSz, fz_);
        fityz = fy_ & fz_;
      }
      const int rc0 = c[0] - tb[0], rc1 = c[1] - tb[1], rc2 = c[2] - tb[2];
      elig = fitx & fityz & (rc0 >= 0) & (rc0 < ts.T[0]) & (rc1 >= 0) & (rc1 < ts.T[1]) & (rc2 >= 0) & (rc2 < ts.T[2]);
      if (elig) {
        code = ((rc0 | (rc1 << 4) | (rc2 << 8)) << 3) | (rc0 % NX);
        extc = ey ? ey : (ez ? 4 + ez : 0);
        R* rr = rec + lane * REC;
        const R fx = -(w * p.jf[0]), fy = -(w * p.jf[1]), fz = -(w * p.jf[2]);
        R px = 0, py = ey == 1 ? dy : R(0), pz = ez == 1 ? dz : R(0);
#pragma unroll
        for (int i = 0; i < NX; ++i) {
          *reinterpret_cast<Pair2<R>*>(rr + W::oAB + 2 * i) =
              Pair2<R>{S0x[i] + half * DSx[i], half * S0x[i] + third * DSx[i]};
          px += DSx[i];
          rr[W::oPX + i] = fx * px;
        }
#pragma unroll
        for (int i = 0; i < NYZ; ++i) {
          *reinterpret_cast<Pair2<R>*>(rr + W::oY + 2 * i) = Pair2<R>{S0y[i], DSy[i]};
          *reinterpret_cast<Pair2<R>*>(rr + W::oZ + 2 * i) = Pair2<R>{S0z[i], DSz[i]};
          py += DSy[i]; pz += DSz[i];
          rr[W::oPY + i] = fy * py;
          rr[W::oPZ + i] = fz * pz;
        }
      }
    }
    __syncwarp();
    // cell by cell (warp-uniform control flow): all particles of this round that share a window
    unsigned rem = __ballot_sync(0xffffffffu, code >= 0);
    while (rem) {
      const int cd = __shfl_sync(0xffffffffu, code, __ffs(rem) - 1);
      const unsigned m = __ballot_sync(0xffffffffu, code == cd);
      rem &= ~m;
      if ((m >> lane) & 1u) s_order[warp][__popc(m & ((1u << lane) - 1u))] = lane;
      __syncwarp();
      const int cnt = __popc(m);
      const int ib = cd >> 3, ph = cd & 7;
      const bool adv = ib == cur + 1;
      JPtr<R> jx_old{};
      if (cur != INT_MIN) jx_old = column(cur);
      if (ib != cur && !adv && cur != INT_MIN) flush_window<R, ORDER, DET>(g, acc, jx_old, curph, grp == 0);
      const int* ord = s_order[warp];
      switch (ph) {
        case 0: cell_batch<R, ORDER, 0, DET>(g, acc, adv, jx_old, grp == 0, rec, ord, cnt, grp, j, k); break;
        case 1: cell_batch<R, ORDER, 1, DET>(g, acc, adv, jx_old, grp == 0, rec, ord, cnt, grp, j, k); break;
        case 2: cell_batch<R, ORDER, 2, DET>(g, acc, adv, jx_old, grp == 0, rec, ord, cnt, grp, j, k); break;
        case 3: cell_batch<R, ORDER, 3 % NX, DET>(g, acc, adv, jx_old, grp == 0, rec, ord, cnt, grp, j, k); break;
        case 4: cell_batch<R, ORDER, 4 % NX, DET>(g, acc, adv, jx_old, grp == 0, rec, ord, cnt, grp, j, k); break;
        default: cell_batch<R, ORDER, 5 % NX, DET>(g, acc, adv, jx_old, grp == 0, rec, ord, cnt, grp, j, k); break;
      }
      cur = ib;
      curph = ph;
      __syncwarp();
    }
    if constexpr (kExt) {
      extra_node_deposit<R, ORDER, DET, W>(g, rec, extc, x1[1], x1[2], w, p.jf, b0 + ((code >> 3) & 15),
                                          b1 + ((code >> 7) & 15), b2 + (code >> 11));
      __syncwarp();
    }
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
  if (cur != INT_MIN) flush_window<R, ORDER, DET>(g, acc, column(cur), curph, grp == 0);
}

// =================================================================== Esirkepov, fp32 order 1: J of the tile in shared memory
// north_star's own design ("accumulates J per tile in shared memory with warp-level reductions and then
// flushes to global memory with atomics"), which fp64 cannot use (64-bit floating-point atomics on shared
// memory are compare-and-swap loops: measured slower in round 1) but fp32 can: RED.shared.f32 is native. At
// order 1 a particle touches 4 x 2 x 2 nodes and has 28 non-zero contributions (Jx 3 x 4, Jy 4 x 2, Jz 4 x 2:
// the last running sum of each axis is zero), few enough for one lane to hold: lane = particle; the 28 x 32
// values of a round are transposed through shared memory, lane l sums value l over every run of same-cell
// particles (the sorted order makes them neighbours) and adds the sums into the tile's J box in shared memory
// (11 x 9 x 9 nodes); the box goes to global memory once per tile, one reduction per non-zero node. The lane-group kernel
// k_deposit_tile needs 46 warp instructions per particle for this case (ncu: issue slots 80 % busy: ballots,
// group shuffles and flushes around 24 FMAs); this one needs about half. Not bit-reproducible from run to run
// (the order of the shared-memory additions is free), so pic_options.deterministic keeps k_deposit_tile.
struct SmemCic {
  static constexpr int BX = 11, BY = 9, BZ = 9;   // nodes tb-1 .. tb+9 along x, tb .. tb+8 along y and z
  static constexpr int PX = 12;                   // padded x extent
  static constexpr int VOL = BZ * BY * PX;
};

__global__ void __launch_bounds__(256, 4)
    k_deposit_smem_cic(Grid<float> g, Particles<float> p, float* __restrict__ xn, float* __restrict__ yn, float* __restrict__ zn,
                       const int32_t* __restrict__ tile_start, TileSpec ts, int32_t* __restrict__ stray_list,
                       unsigned int* __restrict__ stray_count, unsigned long long* deactivated) {
  using R = float;
  using B = SmemCic;
  __shared__ R sJ[3 * B::VOL];
  __shared__ R s_val[8 * 28 * 33];   // per warp: 28 values x 32 particles, row stride 33 (conflict-free both ways)
  __shared__ int s_node[8 * 32];
  const int tile = blockIdx.x;
  const int s = tile_start[tile], e = tile_start[tile + 1];
  if (s >= e) return;
  int tb[3];
  tile_coords(ts, tile, tb);
  for (int i = threadIdx.x; i < 3 * B::VOL; i += blockDim.x) sJ[i] = R(0);
  __syncthreads();
  const int lane = threadIdx.x & 31;
  const R half = R(0.5), third = R(1) / R(3);
  // the box element (relative to the window's first node) that value `lane` of the 28 belongs to
  int my_off = 0;
  if (lane < 12) my_off = lane / 4 + B::PX * ((lane & 1) + B::BY * ((lane >> 1) & 1));
  else if (lane < 20) my_off = B::VOL + (lane - 12) / 2 + B::PX * B::BY * ((lane - 12) & 1);
  else if (lane < 28) my_off = 2 * B::VOL + (lane - 20) / 2 + B::PX * ((lane - 20) & 1);
  for (int base = s; base < e; base += blockDim.x) {   // CTA-uniform trip count: whole warps stay together
    const int t = base + threadIdx.x;
    const bool valid = t < e;
    bool elig = false;
    R x1[3] = {0, 0, 0};
    R w = 0;
    int key = -1 - lane;   // particles that do not take part are runs of their own
    R v[28];
#pragma unroll
    for (int i = 0; i < 28; ++i) v[i] = R(0);
    int node0 = 0;
    if (valid) {
      const R x0[3] = {p.x[t], p.y[t], p.z[t]};
      x1[0] = xn[t]; x1[1] = yn[t]; x1[2] = zn[t];
      w = p.w[t];
      R S0x[4], DSx[4], S0y[2], DSy[2], S0z[2], DSz[2];
      int c[3];
      bool fit[3];
      axis_window<R, 1, 4, 1>(mul_rn(x0[0], g.inv_dx[0]), mul_rn(x1[0], g.inv_dx[0]), c[0], S0x, DSx, fit[0]);
      axis_window<R, 1, 2, 0>(mul_rn(x0[1], g.inv_dx[1]), mul_rn(x1[1], g.inv_dx[1]), c[1], S0y, DSy, fit[1]);
      axis_window<R, 1, 2, 0>(mul_rn(x0[2], g.inv_dx[2]), mul_rn(x1[2], g.inv_dx[2]), c[2], S0z, DSz, fit[2]);
      const int rc0 = c[0] - tb[0], rc1 = c[1] - tb[1], rc2 = c[2] - tb[2];
      elig = fit[0] & fit[1] & fit[2] & (rc0 >= 0) & (rc0 < ts.T[0]) & (rc1 >= 0) & (rc1 < ts.T[1]) & (rc2 >= 0) & (rc2 < ts.T[2]);
      if (elig) {
        key = rc0 | (rc1 << 4) | (rc2 << 8);
        node0 = rc0 + B::PX * (rc1 + B::BY * rc2);   // local node (cell - 1, cell, cell): the window's first node
        const R fx = -(w * p.jf[0]), fy = -(w * p.jf[1]), fz = -(w * p.jf[2]);
        // Jx[i][j][k] = fx (DSx[0] + .. + DSx[i]) (S0z[k] (S0y[j] + DSy[j]/2) + DSz[k] (S0y[j]/2 + DSy[j]/3)), i = 0..2
        R px = 0;
#pragma unroll
        for (int i = 0; i < 3; ++i) {
          px += DSx[i];
#pragma unroll
          for (int k = 0; k < 2; ++k)
#pragma unroll
            for (int j = 0; j < 2; ++j)
              v[4 * i + 2 * k + j] = fx * px * (S0z[k] * (S0y[j] + half * DSy[j]) + DSz[k] * (half * S0y[j] + third * DSy[j]));
        }
        // Jy[i][0][k] = fy DSy[0] (A[i] S0z[k] + B[i] DSz[k]),  Jz[i][j][0] = fz DSz[0] (A[i] S0y[j] + B[i] DSy[j])
#pragma unroll
        for (int i = 0; i < 4; ++i) {
          const R A = S0x[i] + half * DSx[i], Bc = half * S0x[i] + third * DSx[i];
#pragma unroll
          for (int k = 0; k < 2; ++k) v[12 + 2 * i + k] = fy * DSy[0] * (A * S0z[k] + Bc * DSz[k]);
#pragma unroll
          for (int j = 0; j < 2; ++j) v[20 + 2 * i + j] = fz * DSz[0] * (A * S0y[j] + Bc * DSy[j]);
        }
      }
    }
    // runs of equal keys (the sorted order makes same-cell particles neighbours): their 28 sums go to the J box
    const int prev = __shfl_up_sync(0xffffffffu, key, 1);
    const unsigned heads = __ballot_sync(0xffffffffu, lane == 0 || key != prev);
    // transposed through shared memory: lane p stores its 28 values as a column, lane l then walks ROW l over the
    // 32 particles and adds the sum of every run into the box (the run boundaries are warp-uniform): 28 stores +
    // 32 loads per lane. Measured on C3: 0.469 ms; the same sums by a segmented shuffle reduction (28 values x up
    // to 5 steps, head lanes adding) 0.645 ms; every lane adding its own values (8 lanes per address) 1.98 ms
    {
      R* sv = s_val + (threadIdx.x >> 5) * (28 * 33);
      int* sn = s_node + (threadIdx.x >> 5) * 32;
#pragma unroll
      for (int i = 0; i < 28; ++i) sv[i * 33 + lane] = v[i];
      sn[lane] = elig ? node0 : -1;
      __syncwarp();
      const R* row = sv + (lane < 28 ? lane : 0) * 33;
      R acc = 0;
#pragma unroll
      for (int q = 0; q < 32; ++q) {
        acc += row[q];
        if (q == 31 || ((heads >> (q + 1)) & 1u)) {   // warp-uniform
          const int n0 = sn[q];
          if (n0 >= 0 && lane < 28) atomicAdd(sJ + n0 + my_off, acc);
          acc = 0;
        }
      }
      __syncwarp();
    }
    // particles deposited here are finished: wrap and store; the others go to the list untouched
    const bool stray = valid && !elig;
    const unsigned sm = __ballot_sync(0xffffffffu, stray);
    if (sm) {
      unsigned b0 = 0;
      if (lane == 0) b0 = atomicAdd(stray_count, (unsigned)__popc(sm));
      b0 = __shfl_sync(0xffffffffu, b0, 0);
      if (stray) stray_list[b0 + __popc(sm & ((1u << lane) - 1u))] = (int32_t)t;
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
  __syncthreads();
  // the tile's box -> J, one reduction per non-zero node; x fastest, so a warp's reductions are contiguous
  for (int i = threadIdx.x; i < 3 * B::VOL; i += blockDim.x) {
    const R val = sJ[i];
    if (val != R(0)) {
      const int comp = i / B::VOL, r = i % B::VOL;
      const int lx = r % B::PX, ly = (r / B::PX) % B::BY, lz = r / (B::PX * B::BY);
      red_add(g.J[comp] + g.idx(tb[0] - 1 + lx, tb[1] + ly, tb[2] + lz), val);
    }
  }
}

// =================================================================== Esirkepov on the fp64 tensor pipe
// The sums of one cell's particles are small dense contractions over the particles p:
//   Jx[i][jk] += sum_p PX_p[i] * cx_p[jk]
//   Jy[i][jk] += sum_p A_p[i] * (PY_p[j] S0z_p[k]) + B_p[i] * (PY_p[j] DSz_p[k])       (Jz alike)
// with i the NX window nodes along x and jk the NYZ^2 columns, i.e. C[8 x 16] += A[8 x K] B[K x 16]
// with K = particles, four per step (Jy and Jz take two steps each, one per term):
// mma.sync.m8n8k4.f64 (DMMA), ten per four particles, one warp per run of same-cell particles.
// Row r of C holds window node X with X mod 8 == r, so C never moves when the window advances: the
// row of the node that left is reduced into J (one RED per element) and reused.
__device__ __forceinline__ void dmma_884(double& c0, double& c1, double a, double b) {
  asm("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1}, {%2}, {%3}, {%0,%1};"
               : "+d"(c0), "+d"(c1)
               : "d"(a), "d"(b));
}

template <int ORDER>
struct MWin {
  using T = TWin<ORDER>;
  static constexpr int NX = T::NX, BLX = T::BLX, NYZ = T::NYZ, BLYZ = T::BLYZ;
  static constexpr int NCOL = NYZ * NYZ;              // 16 (orders 2, 3) or 4 (order 1)
  static constexpr int NB = NCOL > 8 ? NCOL / 8 : 1;  // 8-column blocks of C
  static constexpr int KSTEP = NYZ == 4 ? 2 : 0;      // k advances by this from one column block to the next
  // record (elements): {A_x,B_x}[NX] | PX[NX] | {S0_y,DS_y}[NYZ] | PY[NYZ] | {S0_z,DS_z}[NYZ] | PZ[NYZ]
  static constexpr int oAB = 0, oPX = 2 * NX, oY = 3 * NX, oPY = oY + 2 * NYZ, oZ = oPY + NYZ, oPZ = oZ + 2 * NYZ;
  static constexpr int RAW = oPZ + NYZ;                            // 42 / 24
  static constexpr int REC = (RAW / 2) % 2 == 1 ? RAW : RAW + 2;   // REC/2 odd: conflict-free pair stores
};

// C fragments of one lane: rows = window nodes (lane >> 2), columns 2*(lane & 3) + {0,1} of each block
template <int NB>
struct CFrag {
  double x[NB][2], y[NB][2], z[NB][2];
  __device__ __forceinline__ void zero() {
#pragma unroll
    for (int b = 0; b < NB; ++b)
#pragma unroll
      for (int e = 0; e < 2; ++e) { x[b][e] = 0; y[b][e] = 0; z[b][e] = 0; }
  }
};

template <class R, int ORDER, int NWARP, int MINB, int DET>
__global__ void __launch_bounds__(NWARP * 32, MINB)
    k_deposit_mma(Grid<R> g, Particles<R> p, R* __restrict__ xn, R* __restrict__ yn, R* __restrict__ zn,
                  const int32_t* __restrict__ tile_start, TileSpec ts, int32_t* __restrict__ stray_list,
                  unsigned int* __restrict__ stray_count, unsigned long long* deactivated) {
  using W = MWin<ORDER>;
  constexpr int NX = W::NX, NYZ = W::NYZ, NB = W::NB, REC = W::REC, BLX = W::BLX, BLYZ = W::BLYZ;
  extern __shared__ __align__(128) unsigned char smem_raw[];
  R* rec_all = reinterpret_cast<R*>(smem_raw);
  __shared__ unsigned char s_ord[NWARP][32];   // record slots of the group being contracted, in order

  const int tile = blockIdx.x;
  const int s = tile_start[tile], e = tile_start[tile + 1];
  if (s >= e) return;
  int tb[3];
  tile_coords(ts, tile, tb);

  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  const int gq = lane >> 2, t = lane & 3;           // fragment coordinates of this lane
  R* rec = rec_all + (size_t)warp * 33 * REC;       // 32 records of the round + one that stays zero
  const R* zrec = rec + 32 * REC;
  for (int i = lane; i < REC; i += 32) rec[32 * REC + i] = R(0);
  const R half = R(0.5), third = R(1) / R(3);

  // B operands: this lane supplies column gq (+ 8 per block) = (jB, kB + KSTEP * block)
  const bool colok = gq < W::NCOL;
  const int jB = colok ? gq % NYZ : 0, kB = colok ? gq / NYZ : 0;
  const int offY = W::oY + 2 * jB, offPY = W::oPY + jB, offZ = W::oZ + 2 * kB,
            offPZ = W::oPZ + kB;
  // C fragments: this lane holds columns 2t + {0,1} (+ 8 per block) of row gq
  int coff[NB][2];
  bool cok[NB][2];
#pragma unroll
  for (int b = 0; b < NB; ++b)
#pragma unroll
    for (int c = 0; c < 2; ++c) {
      const int n = 2 * t + c + 8 * b;
      cok[b][c] = n < W::NCOL;
      coff[b][c] = (n % NYZ) * g.sy + (n / NYZ) * g.sz;
    }

  CFrag<NB> C;
  C.zero();
  int cur = INT_MIN;   // packed cell triple of the window being accumulated
  auto win_x = [&](int cd) { return tb[0] + 3 * (cd & 15) - 4 - BLX; };   // first node of a triple's 8-node window
  auto win_y = [&](int cd) { return tb[1] + ((cd >> 4) & 15) - 4 - BLYZ; };
  auto win_z = [&](int cd) { return tb[2] + (cd >> 8) - 4 - BLYZ; };
  // rows of the old window that the new one (nx0 .. nx0+7 on the same y,z; none if !same_row) does
  // not contain go to J, one reduction per element, and are cleared
  auto retire_rows = [&](bool same_row, int nx0) {
    const int ox0 = win_x(cur);
    const int io = (gq - ox0) & 7;
    const int X = ox0 + io;
    const bool keep = same_row && X >= nx0 && X < nx0 + 8;
    if (!keep) {
      const int base = g.idx(X, win_y(cur), win_z(cur));
#pragma unroll
      for (int b = 0; b < NB; ++b)
#pragma unroll
        for (int c = 0; c < 2; ++c) {
          if (cok[b][c]) {
            if (C.x[b][c] != 0.0) j_add<R, DET>(g, g.J[0] + base + coff[b][c], (R)C.x[b][c]);
            if (C.y[b][c] != 0.0) j_add<R, DET>(g, g.J[1] + base + coff[b][c], (R)C.y[b][c]);
            if (C.z[b][c] != 0.0) j_add<R, DET>(g, g.J[2] + base + coff[b][c], (R)C.z[b][c]);
          }
          C.x[b][c] = 0; C.y[b][c] = 0; C.z[b][c] = 0;
        }
    }
  };

  // the warp's contiguous share of the tile, a multiple of 32 particles; gridDim.y CTAs share a tile when the
  // grid has too few tiles to fill the machine (C1: 8 tiles)
  const int n = e - s;
  const int vwarps = NWARP * (int)gridDim.y;
  const int chunk = ((n + vwarps - 1) / vwarps + 31) & ~31;
  const int wb = min(e, s + ((int)blockIdx.y * NWARP + warp) * chunk);
  const int we = min(e, wb + chunk);

  for (int rb = wb; rb < we; rb += 32) {
    const int tp = rb + lane;
    const bool valid = tp < we;
    bool elig = false;
    R x1[3] = {0, 0, 0};
    R w = 0;
    int code = -1;
    int extc = 0;           // extra node of a particle that crossed a face in y or z (extra_node_deposit)
    if (tp + 32 < we) {   // the next round's particle data on its way to L2 while this round computes
      prefetch_l2(p.x + tp + 32); prefetch_l2(p.y + tp + 32); prefetch_l2(p.z + tp + 32);
      prefetch_l2(xn + tp + 32); prefetch_l2(yn + tp + 32); prefetch_l2(zn + tp + 32);
      prefetch_l2(p.w + tp + 32);
    }
    if (valid) {
      R x0[3] = {p.x[tp], p.y[tp], p.z[tp]};
      x1[0] = xn[tp]; x1[1] = yn[tp]; x1[2] = zn[tp];
      w = p.w[tp];
      int c[3];
      int ec;
      const bool fits = build_record<R, ORDER, W>(g, p.jf, rec + lane * REC, x0, x1, w, c, ec);
      // the cell must be inside the grid and within 4 cells of the tile (4-bit biased offsets)
      const int rc0 = c[0] - tb[0] + 4, rc1 = c[1] - tb[1] + 4, rc2 = c[2] - tb[2] + 4;
      elig = fits & (((rc0 | rc1 | rc2) & ~15) == 0) & (c[0] >= 0) & (c[0] < g.N[0]) & (c[1] >= 0) & (c[1] < g.N[1]) &
             (c[2] >= 0) & (c[2] < g.N[2]);
      if (elig) {
        code = rc0 | (rc1 << 4) | (rc2 << 8);
        extc = ec;
      }
    }
    __syncwarp();
    // groups of particles of this round whose cells lie in the same triple of x-neighbouring cells of one
    // (y,z) row: their windows span 8 nodes together, exactly the 8 rows of C, so they share the
    // accumulators (fewer padded contraction steps, and three rows retire at once). The groups are formed
    // over the whole round, not over consecutive particles: in a hot plasma the order is stale between two
    // sorts, and every particle out of place would otherwise end a run and send the accumulated rows to J
    // (C5: L2 at 69 % with reductions). The triple being accumulated goes first. Warp-uniform control flow.
    const int scode = code < 0 ? -1 : ((code & ~15) | ((code & 15) / 3));
    unsigned rem = __ballot_sync(0xffffffffu, code >= 0);
    while (rem) {
      unsigned m = cur != INT_MIN ? (__ballot_sync(0xffffffffu, scode == cur) & rem) : 0u;
      int cd = cur;
      if (m == 0) {
        cd = __shfl_sync(0xffffffffu, scode, __ffs(rem) - 1);
        m = __ballot_sync(0xffffffffu, scode == cd);
      }
      rem &= ~m;
      if ((m >> lane) & 1u) s_ord[warp][__popc(m & ((1u << lane) - 1u))] = (unsigned char)lane;
      __syncwarp();
      const int cnt = __popc(m);
      if (cd != cur) {
        if (cur != INT_MIN) retire_rows(((cd ^ cur) >> 4) == 0, win_x(cd));
        cur = cd;
      }
#ifndef PIC_X_UNROLL
#define PIC_X_UNROLL 2
#endif
      constexpr int kUnrollSteps = PIC_X_UNROLL;
#pragma unroll kUnrollSteps
      for (int b = 0; b < cnt; b += 4) {
        // four particles per contraction step, K = particle: this lane supplies, for the group's particle
        // b + t, the A operands of its row (a node of that particle's own 6-node window, or zero) and the
        // B operands of its column(s)
        const bool here = b + t < cnt;
        const int src = here ? (int)s_ord[warp][b + t] : 32;          // slot 32: the all-zero record
        const int pc = __shfl_sync(0xffffffffu, code, src & 31);
        const int i = (gq - (tb[0] + (pc & 15) - 4 - BLX)) & 7;      // window slot of this lane's row
        const bool rowok = i < NX;
        const R* rr = rec + src * REC;
        const R* ra = rowok ? rr : zrec;
        const double px = ra[W::oPX + (rowok ? i : 0)];
        const Pair2<R> ab = *reinterpret_cast<const Pair2<R>*>(ra + W::oAB + 2 * (rowok ? i : 0));
        const Pair2<R> yv = *reinterpret_cast<const Pair2<R>*>(rr + offY);
        const double py = colok ? (double)rr[offPY] : 0.0;
        const double y0 = colok ? (double)yv.a : 0.0, y1 = colok ? (double)yv.b : 0.0;
        const double al = fma(0.5, y1, y0), be = fma(0.5, y0, y1 * (1.0 / 3.0));
#pragma unroll
        for (int nb = 0; nb < NB; ++nb) {
          const Pair2<R> zv = *reinterpret_cast<const Pair2<R>*>(rr + offZ + 2 * W::KSTEP * nb);
          const double pz = rr[offPZ + W::KSTEP * nb];
          const double z0 = zv.a, z1 = zv.b;
          dmma_884(C.x[nb][0], C.x[nb][1], px, fma(z0, al, z1 * be));
          dmma_884(C.y[nb][0], C.y[nb][1], (double)ab.a, py * z0);
          dmma_884(C.z[nb][0], C.z[nb][1], (double)ab.a, pz * y0);
          dmma_884(C.y[nb][0], C.y[nb][1], (double)ab.b, py * z1);
          dmma_884(C.z[nb][0], C.z[nb][1], (double)ab.b, pz * y1);
        }
      }
      __syncwarp();   // s_ord is rewritten by the next group
    }
    extra_node_deposit<R, ORDER, DET, W>(g, rec, extc, x1[1], x1[2], w, p.jf, tb[0] + (code & 15) - 4 - BLX,
                                         tb[1] + ((code >> 4) & 15) - 4 - BLYZ, tb[2] + (code >> 8) - 4 - BLYZ);
    __syncwarp();
    // particles deposited here are finished: wrap and store; the others go to the list untouched
    const bool stray = valid && !elig;
    const unsigned sm = __ballot_sync(0xffffffffu, stray);
    if (sm) {
      unsigned base = 0;
      if (lane == 0) base = atomicAdd(stray_count, (unsigned)__popc(sm));
      base = __shfl_sync(0xffffffffu, base, 0);
      if (stray) stray_list[base + __popc(sm & ((1u << lane) - 1u))] = (int32_t)tp;
    }
    if (valid && elig) {
      bool out = false;
#pragma unroll
      for (int d = 0; d < 3; ++d) out |= wrap_axis<R>(x1[d], g.L[d], g.periodic[d]);
      if (out) {
        if (w != R(0)) atomicAdd(deactivated, 1ull);
        p.w[tp] = R(0);
      }
      xn[tp] = x1[0]; yn[tp] = x1[1]; zn[tp] = x1[2];
    }
  }
  if (cur != INT_MIN) retire_rows(false, 0);
}

// =================================================================== gather + push + deposit, one kernel (fp64)
// PAPER.md:114 argues for fusing the gather into the push so that no per-particle field ever reaches
// memory; the same argument holds one step further: the deposit needs x_old, x_new, w and the nodal
// weights of x_old, all of which the push has in registers. Here one CTA per tile stages the E/B box
// (as k_push_tile) and each warp takes rounds of 32 particles through the whole particle step: lane =
// particle for gather + push + the deposit's per-axis record, then the warp contracts the round's records
// on the fp64 tensor pipe (as k_deposit_mma). x_new goes to memory once, wrapped; x_old, w and the record
// never do. The gather is bound by shared-memory wavefronts and the contraction by the fp64 pipe, so warps
// in different phases of their rounds fill each other's idle unit on the same SM.
// Particles that drifted out of the tile's box since the last sort are listed and taken through the same
// code in a second pass that gathers from global memory (all lanes busy); particles whose move does not
// fit the deposit windows (cell change in y or z) are pushed here and listed for k_deposit_list_warp.
template <int ORDER, int PUSHER, int GATHER, int NWARP>
__global__ void __launch_bounds__(NWARP * 32, 1)
    k_fused_mma(Grid<double> g, Particles<double> p, double* __restrict__ xn, double* __restrict__ yn,
                double* __restrict__ zn, const int32_t* __restrict__ tile_start, TileSpec ts,
                int32_t* __restrict__ stray_list, unsigned int* __restrict__ stray_count,
                unsigned long long* deactivated) {
  using R = double;
  using PB = PushBox<ORDER>;
  using W = MWin<ORDER>;
  constexpr int E = PB::EXT, SX = PB::SX, VOL = PB::VOL;
  constexpr int NS = GATHER == 1 ? ORDER : ORDER + 1;   // weights along a staggered axis
  constexpr int NN = ORDER + 1;
  constexpr int NX = W::NX, NYZ = W::NYZ, NB = W::NB, REC = W::REC, BLX = W::BLX, BLYZ = W::BLYZ;
  constexpr int MAXD = kFusedMaxDrift;
  extern __shared__ __align__(128) unsigned char smem_raw[];
  R* box = reinterpret_cast<R*>(smem_raw);   // [6][E (x)][SX: E (z) x E (y), padded]
  R* rec_all = box + 6 * VOL;
  __shared__ int s_drift[NWARP][MAXD];   // per warp, in processing order: nothing here depends on timing

  const int tile = blockIdx.x;
  const int s = tile_start[tile], e = tile_start[tile + 1];
  if (s >= e) return;
  int tb[3];
  tile_coords(ts, tile, tb);
  const int o0 = tb[0] - PB::HB, o1 = tb[1] - PB::HB, o2 = tb[2] - PB::HB;   // node of local (0,0,0)
  {
    const int lim0 = g.N[0] + kGuard, lim1 = g.N[1] + kGuard, lim2 = g.N[2] + kGuard;
    for (int idx = threadIdx.x; idx < E * E * E; idx += blockDim.x) {
      int i = idx % E, r = idx / E;
      int j = r % E, k = r / E;
      const bool in = (o0 + i < lim0) & (o1 + j < lim1) & (o2 + k < lim2);
      const int gi = g.idx(o0 + i, o1 + j, o2 + k);
      const int li = SX * i + j + E * k;
#pragma unroll
      for (int c = 0; c < 6; ++c) {
        if (in) cp_async(box + c * VOL + li, g.F[c] + gi);
        else box[c * VOL + li] = R(0);
      }
    }
  }

  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  const int gq = lane >> 2, t = lane & 3;           // fragment coordinates of this lane
  R* rec = rec_all + (size_t)warp * 33 * REC;       // 32 records of the round + one that stays zero
  const R* zrec = rec + 32 * REC;
  for (int i = lane; i < REC; i += 32) rec[32 * REC + i] = R(0);
  const R half = R(0.5), third = R(1) / R(3);

  // B operands: this lane supplies column gq (+ 8 per block) = (jB, kB + KSTEP * block)
  const bool colok = gq < W::NCOL;
  const int jB = colok ? gq % NYZ : 0, kB = colok ? gq / NYZ : 0;
  const int offY = W::oY + 2 * jB, offPY = W::oPY + jB, offZ = W::oZ + 2 * kB, offPZ = W::oPZ + kB;
  // C fragments: this lane holds columns 2t + {0,1} (+ 8 per block) of row gq
  int coff[NB][2];
  bool cok[NB][2];
#pragma unroll
  for (int b = 0; b < NB; ++b)
#pragma unroll
    for (int c = 0; c < 2; ++c) {
      const int n = 2 * t + c + 8 * b;
      cok[b][c] = n < W::NCOL;
      coff[b][c] = (n % NYZ) * g.sy + (n / NYZ) * g.sz;
    }

  CFrag<NB> C;
  C.zero();
  int cur = INT_MIN;   // packed cell triple of the window being accumulated
  auto win_x = [&](int cd) { return tb[0] + 3 * (cd & 15) - 4 - BLX; };   // first node of a triple's 8-node window
  auto win_y = [&](int cd) { return tb[1] + ((cd >> 4) & 15) - 4 - BLYZ; };
  auto win_z = [&](int cd) { return tb[2] + (cd >> 8) - 4 - BLYZ; };
  auto retire_rows = [&](bool same_row, int nx0) {
    const int ox0 = win_x(cur);
    const int io = (gq - ox0) & 7;
    const int X = ox0 + io;
    const bool keep = same_row && X >= nx0 && X < nx0 + 8;
    if (!keep) {
      const int base = g.idx(X, win_y(cur), win_z(cur));
#pragma unroll
      for (int b = 0; b < NB; ++b)
#pragma unroll
        for (int c = 0; c < 2; ++c) {
          if (cok[b][c]) {
            if (C.x[b][c] != 0.0) j_add<R>(g, g.J[0] + base + coff[b][c], C.x[b][c]);
            if (C.y[b][c] != 0.0) j_add<R>(g, g.J[1] + base + coff[b][c], C.y[b][c]);
            if (C.z[b][c] != 0.0) j_add<R>(g, g.J[2] + base + coff[b][c], C.z[b][c]);
          }
          C.x[b][c] = 0; C.y[b][c] = 0; C.z[b][c] = 0;
        }
    }
  };

  // the warp's contiguous share of the tile: whole rounds of 32, sizes differing by at most one round
  const int n = e - s;
  const int rounds = (n + 31) >> 5;
  const int wb = s + 32 * (int)(((long long)rounds * warp) / NWARP);
  const int we = min(e, s + 32 * (int)(((long long)rounds * (warp + 1)) / NWARP));

  asm volatile("cp.async.wait_all;" ::: "memory");
  __syncthreads();

  int ndrift = 0;   // entries of this warp's list (warp-uniform)
#pragma unroll 1
  for (int phase = 0; phase < 2; ++phase) {
    int r_begin = wb, r_end = we;
    if (phase == 1) {
      __syncwarp();
      r_begin = 0;
      r_end = ndrift;
    }
#pragma unroll 1
    for (int rb = r_begin; rb < r_end; rb += 32) {
      bool valid = rb + lane < r_end;
      int tp = rb + lane;
      if (phase == 1) tp = valid ? s_drift[warp][tp] : 0;
      bool elig = false;
      R x1[3] = {0, 0, 0};
      R w = 0;
      int code = -1;
      if (phase == 0 && tp + 32 < we) {   // the next round's particle data on its way to L2
        prefetch_l2(p.x + tp + 32); prefetch_l2(p.y + tp + 32); prefetch_l2(p.z + tp + 32);
        prefetch_l2(p.ux + tp + 32); prefetch_l2(p.uy + tp + 32); prefetch_l2(p.uz + tp + 32);
        prefetch_l2(p.w + tp + 32);
      }
      R x0[3], u[3], wn[3][ORDER + 1], xi0[3], Ef[3], Bf[3];
      int ln[3];
      bool drifted = false;
      if (valid) {
        x0[0] = p.x[tp]; x0[1] = p.y[tp]; x0[2] = p.z[tp];
        u[0] = p.ux[tp]; u[1] = p.uy[tp]; u[2] = p.uz[tp];
        w = p.w[tp];
        bool inbox = phase == 0;
        {
          R ws[3][ORDER + 1];
          int ls[3];
#pragma unroll
          for (int d = 0; d < 3; ++d) {
            xi0[d] = mul_rn(x0[d], g.inv_dx[d]);
            const R xs = sub_rn(xi0[d], R(0.5));
            const int od = d == 0 ? o0 : (d == 1 ? o1 : o2);
            ln[d] = shape<R, ORDER>(xi0[d], wn[d]);
            ls[d] = (GATHER == 1 ? shape_lowered<R, ORDER>(xs, ws[d]) : shape<R, ORDER>(xs, ws[d])) - od;
            const int lr = ln[d] - od;
            inbox &= (lr >= 0) & (lr <= E - ORDER - 1) & (ls[d] >= 0) & (ls[d] <= E - ORDER - 1);
          }
          if (inbox) {
            const int l0 = ln[0] - o0, l1 = ln[1] - o1, l2 = ln[2] - o2;
            // Ex (s,n,n)  Ey (n,s,n)  Ez (n,n,s)  Bx (n,s,s)  By (s,n,s)  Bz (s,s,n)
            Ef[0] = interp_box<R, ORDER, false, NS, NN, NN>(box + 0 * VOL, SX * ls[0] + l1 + E * l2, ws[0], wn[1], wn[2]);
            Ef[1] = interp_box<R, ORDER, false, NN, NS, NN>(box + 1 * VOL, SX * l0 + ls[1] + E * l2, wn[0], ws[1], wn[2]);
            Ef[2] = interp_box<R, ORDER, false, NN, NN, NS>(box + 2 * VOL, SX * l0 + l1 + E * ls[2], wn[0], wn[1], ws[2]);
            Bf[0] = interp_box<R, ORDER, false, NN, NS, NS>(box + 3 * VOL, SX * l0 + ls[1] + E * ls[2], wn[0], ws[1], ws[2]);
            Bf[1] = interp_box<R, ORDER, false, NS, NN, NS>(box + 4 * VOL, SX * ls[0] + l1 + E * ls[2], ws[0], wn[1], ws[2]);
            Bf[2] = interp_box<R, ORDER, false, NS, NS, NN>(box + 5 * VOL, SX * ls[0] + ls[1] + E * l2, ws[0], ws[1], wn[2]);
          }
        }
        drifted = !inbox;
      }
      // drifted out of the tile's box since the last sort: listed (per warp, in order) for the second pass,
      // which gathers from global memory with all lanes busy; in line if the list is full
      if (phase == 0) {
        const unsigned dm = __ballot_sync(0xffffffffu, drifted);
        if (dm) {
          const int slot = ndrift + __popc(dm & ((1u << lane) - 1u));
          if (drifted && slot < MAXD) {
            s_drift[warp][slot] = tp;
            valid = false;
          }
          ndrift = min(MAXD, ndrift + __popc(dm));
        }
      }
      if (valid) {
        if (drifted) gather6<R, ORDER, GATHER != 0>(g, x0[0], x0[1], x0[2], Ef, Bf);
        {
          push_momentum<R>(PUSHER, p.kq, g.inv_c2, Ef, Bf, u);
          advance<R>(g.dt, g.inv_c2, x0, u, x1);
          p.ux[tp] = u[0]; p.uy[tp] = u[1]; p.uz[tp] = u[2];
          R S0x[NX], DSx[NX], S0y[NYZ], DSy[NYZ], S0z[NYZ], DSz[NYZ];
          int c[3];
          bool fit[3];
          axis_window_from<R, ORDER, NX, BLX>(ln[0], wn[0], xi0[0], mul_rn(x1[0], g.inv_dx[0]), c[0], S0x, DSx, fit[0]);
          axis_window_from<R, ORDER, NYZ, BLYZ>(ln[1], wn[1], xi0[1], mul_rn(x1[1], g.inv_dx[1]), c[1], S0y, DSy, fit[1]);
          axis_window_from<R, ORDER, NYZ, BLYZ>(ln[2], wn[2], xi0[2], mul_rn(x1[2], g.inv_dx[2]), c[2], S0z, DSz, fit[2]);
          // the cell must be inside the grid and within 4 cells of the tile (4-bit biased offsets)
          const int rc0 = c[0] - tb[0] + 4, rc1 = c[1] - tb[1] + 4, rc2 = c[2] - tb[2] + 4;
          elig = fit[0] & fit[1] & fit[2] & (((rc0 | rc1 | rc2) & ~15) == 0) & (c[0] >= 0) & (c[0] < g.N[0]) &
                 (c[1] >= 0) & (c[1] < g.N[1]) & (c[2] >= 0) & (c[2] < g.N[2]);
          if (elig) {
            code = rc0 | (rc1 << 4) | (rc2 << 8);
            R* rr = rec + lane * REC;
            const R fx = -(w * p.jf[0]), fy = -(w * p.jf[1]), fz = -(w * p.jf[2]);
            R px = 0, py = 0, pz = 0;
#pragma unroll
            for (int i = 0; i < NX; ++i) {
              *reinterpret_cast<Pair2<R>*>(rr + W::oAB + 2 * i) =
                  Pair2<R>{S0x[i] + half * DSx[i], half * S0x[i] + third * DSx[i]};
              px += DSx[i];
              rr[W::oPX + i] = fx * px;
            }
#pragma unroll
            for (int i = 0; i < NYZ; ++i) {
              *reinterpret_cast<Pair2<R>*>(rr + W::oY + 2 * i) = Pair2<R>{S0y[i], DSy[i]};
              *reinterpret_cast<Pair2<R>*>(rr + W::oZ + 2 * i) = Pair2<R>{S0z[i], DSz[i]};
              py += DSy[i]; pz += DSz[i];
              rr[W::oPY + i] = fy * py;
              rr[W::oPZ + i] = fz * pz;
            }
          }
        }
      }
      __syncwarp();
      // runs of consecutive particles whose cells lie in the same triple of x-neighbouring cells of one
      // (y,z) row share the accumulators (see k_deposit_mma). Warp-uniform control flow.
      const int scode = code < 0 ? -1 : ((code & ~15) | ((code & 15) / 3));
      const int prev = __shfl_up_sync(0xffffffffu, scode, 1);
      unsigned heads = __ballot_sync(0xffffffffu, lane == 0 || scode != prev);
      const unsigned live = __ballot_sync(0xffffffffu, code >= 0);
      while (heads) {
        const int s0 = __ffs(heads) - 1;
        heads &= heads - 1;
        const int s1 = heads ? __ffs(heads) - 1 : 32;
        if (!((live >> s0) & 1u)) continue;
        const int cd = __shfl_sync(0xffffffffu, scode, s0);
        if (cd != cur) {
          if (cur != INT_MIN) retire_rows(((cd ^ cur) >> 4) == 0, win_x(cd));
          cur = cd;
        }
#pragma unroll 2
        for (int b = s0; b < s1; b += 4) {
          const bool here = b + t < s1;
          const int pc = __shfl_sync(0xffffffffu, code, (b + t) & 31);
          const int i = (gq - (tb[0] + (pc & 15) - 4 - BLX)) & 7;      // window slot of this lane's row
          const bool rowok = i < NX;
          const R* rr = rec + (here ? b + t : 32) * REC;               // slot 32: the all-zero record
          const R* ra = rowok ? rr : zrec;
          const double px = ra[W::oPX + (rowok ? i : 0)];
          const Pair2<R> ab = *reinterpret_cast<const Pair2<R>*>(ra + W::oAB + 2 * (rowok ? i : 0));
          const Pair2<R> yv = *reinterpret_cast<const Pair2<R>*>(rr + offY);
          const double py = colok ? (double)rr[offPY] : 0.0;
          const double y0 = colok ? (double)yv.a : 0.0, y1 = colok ? (double)yv.b : 0.0;
          const double al = fma(0.5, y1, y0), be = fma(0.5, y0, y1 * (1.0 / 3.0));
#pragma unroll
          for (int nb = 0; nb < NB; ++nb) {
            const Pair2<R> zv = *reinterpret_cast<const Pair2<R>*>(rr + offZ + 2 * W::KSTEP * nb);
            const double pz = rr[offPZ + W::KSTEP * nb];
            const double z0 = zv.a, z1 = zv.b;
            dmma_884(C.x[nb][0], C.x[nb][1], px, fma(z0, al, z1 * be));
            dmma_884(C.y[nb][0], C.y[nb][1], (double)ab.a, py * z0);
            dmma_884(C.z[nb][0], C.z[nb][1], (double)ab.a, pz * y0);
            dmma_884(C.y[nb][0], C.y[nb][1], (double)ab.b, py * z1);
            dmma_884(C.z[nb][0], C.z[nb][1], (double)ab.b, pz * y1);
          }
        }
      }
      __syncwarp();
      // particles deposited here are finished: wrap and store; the others are stored unwrapped and listed
      const bool stray = valid && !elig;
      const unsigned sm = __ballot_sync(0xffffffffu, stray);
      if (sm) {
        unsigned base = 0;
        if (lane == 0) base = atomicAdd(stray_count, (unsigned)__popc(sm));
        base = __shfl_sync(0xffffffffu, base, 0);
        if (stray) stray_list[base + __popc(sm & ((1u << lane) - 1u))] = (int32_t)tp;
      }
      if (valid) {
        if (elig) {
          bool out = false;
#pragma unroll
          for (int d = 0; d < 3; ++d) out |= wrap_axis<R>(x1[d], g.L[d], g.periodic[d]);
          if (out) {
            if (w != R(0)) atomicAdd(deactivated, 1ull);
            p.w[tp] = R(0);
          }
        }
        xn[tp] = x1[0]; yn[tp] = x1[1]; zn[tp] = x1[2];
      }
    }
  }
  if (cur != INT_MIN) retire_rows(false, 0);
}

}  // namespace

// >48 KB of dynamic shared memory is an opt-in per function AND per device/context: done once per
// simulation handle (Ctx), not once per process
template <class K>
static void opt_in_smem(Ctx& c, K kernel, size_t bytes) {
  if (c.smem_opted.insert((const void*)kernel).second)
    cudaFuncSetAttribute(kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)bytes);
}

template <int ORDER>
static void launch_fused(const Grid<double>& g, const ParticleStep<double>& a, Ctx& c) {
  const Particles<double>& p = a.cur;
  const int n_tiles = a.tiles.nt[0] * a.tiles.nt[1] * a.tiles.nt[2];
  constexpr int NW = kFusedWarps;
  const size_t smem = ((size_t)6 * PushBox<ORDER>::VOL + (size_t)NW * 33 * MWin<ORDER>::REC) * sizeof(double);
  auto k = g.pusher == 0 ? (g.gather_mode == 0 ? k_fused_mma<ORDER, 0, 0, NW> : k_fused_mma<ORDER, 0, 1, NW>)
                         : (g.gather_mode == 0 ? k_fused_mma<ORDER, 1, 0, NW> : k_fused_mma<ORDER, 1, 1, NW>);
  opt_in_smem(c, k, smem);
  ScopedPhase ph(c, kPhasePush);
  k<<<n_tiles, NW * 32, smem, c.stream>>>(g, p, a.alt.x, a.alt.y, a.alt.z, a.tile_start, a.tiles, a.stray_list,
                                           a.stray_count, a.deactivated);
  c.launches += 1;
}

template <class R, int ORDER>
static void launch_tile_order(const Grid<R>& g, const ParticleStep<R>& a, int mode, Ctx& c) {
  if constexpr (sizeof(R) == 8) {
    if (mode == kDepositFused) { launch_fused<ORDER>(g, a, c); return; }
  }
  const bool mma = mode == kDepositTileMma;
  const Particles<R>& p = a.cur;
  R *xn = a.alt.x, *yn = a.alt.y, *zn = a.alt.z;
  const int n_tiles = a.tiles.nt[0] * a.tiles.nt[1] * a.tiles.nt[2];
  constexpr int kW = kDepTileWarps;
  const bool det = g.fix_scale[0] != 0.0;
  auto kvec = det ? k_deposit_tile<R, ORDER, kW, 1> : k_deposit_tile<R, ORDER, kW, 0>;
  auto kmma = det ? k_deposit_mma<R, ORDER, kDepMmaWarps, kDepMmaCtas, 1> : k_deposit_mma<R, ORDER, kDepMmaWarps, kDepMmaCtas, 0>;
  constexpr int mw = kDepMmaWarps;
  const bool tma = c.tma_push;
  constexpr int ES = (int)sizeof(R);
  const size_t push_smem = (size_t)6 * (tma ? PushBox<ORDER, true, ES>::VOL : PushBox<ORDER, false, ES>::VOL) * sizeof(R);
  const size_t vec_smem = (size_t)kW * 32 * TWin<ORDER>::REC * sizeof(R);
  const size_t mma_smem = (size_t)mw * 33 * MWin<ORDER>::REC * sizeof(R);
  {
    ScopedPhase ph(c, kPhasePush);
    auto pick = [&](auto tma_tag) {
      constexpr bool T = decltype(tma_tag)::value;
      return g.pusher == 0 ? (g.gather_mode == 0 ? k_push_tile<R, ORDER, 0, 0, T> : k_push_tile<R, ORDER, 0, 1, T>)
                           : (g.gather_mode == 0 ? k_push_tile<R, ORDER, 1, 0, T> : k_push_tile<R, ORDER, 1, 1, T>);
    };
    auto kpush = tma ? pick(std::true_type{}) : pick(std::false_type{});
    opt_in_smem(c, kpush, push_smem);
    kpush<<<n_tiles, kPushTileThreads<R>, push_smem, c.stream>>>(g, p, xn, yn, zn, a.tile_start, a.tiles, c.tmap_push);
  }
  {
    ScopedPhase ph(c, kPhaseDeposit);
    if (mma) {
      opt_in_smem(c, kmma, mma_smem);
      // small grids: several CTAs per tile, so that about two waves of CTAs exist
      int split = 1;
      while (split < 8 && (int64_t)n_tiles * split * 2 <= (int64_t)c.sm_count * kDepMmaCtas) split *= 2;
      kmma<<<dim3(n_tiles, split), mw * 32, mma_smem, c.stream>>>(g, p, xn, yn, zn, a.tile_start, a.tiles, a.stray_list,
                                                                 a.stray_count, a.deactivated);
    } else {
      bool smem_cic = false;
      if constexpr (sizeof(R) == 4 && ORDER == 1) {
        // fp32, order 1, floating-point reductions: the tile's J in shared memory (AUTO's choice; mode TILE given
        // explicitly keeps the lane-group kernel)
        if (!det && c.auto_deposit) {
          smem_cic = true;
          k_deposit_smem_cic<<<n_tiles, 256, 0, c.stream>>>(g, p, xn, yn, zn, a.tile_start, a.tiles, a.stray_list,
                                                            a.stray_count, a.deactivated);
        }
      }
      if (!smem_cic) {
        opt_in_smem(c, kvec, vec_smem);
        kvec<<<n_tiles, kW * 32, vec_smem, c.stream>>>(g, p, xn, yn, zn, a.tile_start, a.tiles, a.stray_list,
                                                      a.stray_count, a.deactivated);
      }
    }
  }
  c.launches += 2;
}

// The six E/B arrays are one allocation of six padded boxes (pic_api.cu), i.e. a 4-D tensor (x, y, z,
// component) with x contiguous. TMA needs every stride to be a multiple of 16 bytes and the base 16-byte
// aligned; grids that do not meet that (odd padded extents, odd tiles) keep the cp.async staging.
template <class R>
bool make_push_tensor_map(const Grid<R>& g, int order, int tile_x, int stage_mode, Ctx& c) {
  c.tma_push = false;
  if (stage_mode == 1) return false;                       // PIC_STAGE_CP_ASYNC
  if ((tile_x * sizeof(R)) % 16) return false;             // every box must start at a 16-byte aligned x
  // fp32: only on request. Measured on C3 (order 1): push 0.405 ms with TMA against 0.396 ms with cp.async —
  // the box is small (10^3 nodes of 4 bytes) and the y-fastest layout has slightly fewer bank conflicts there.
  if (sizeof(R) != 8 && stage_mode != 2) return false;
  const size_t es = sizeof(R);
  const size_t st1 = (size_t)g.P[0] * es, st2 = st1 * g.P[1], st3 = st2 * g.P[2];
  if (st1 % 16 || st2 % 16 || st3 % 16 || ((uintptr_t)g.F[0] % 16)) return false;
  for (int k = 1; k < 6; ++k)
    if (g.F[k] != g.F[0] + (size_t)k * (st3 / es)) return false;
  typedef CUresult (*EncodeFn)(CUtensorMap*, CUtensorMapDataType, cuuint32_t, void*, const cuuint64_t*, const cuuint64_t*,
                               const cuuint32_t*, const cuuint32_t*, CUtensorMapInterleave, CUtensorMapSwizzle,
                               CUtensorMapL2promotion, CUtensorMapFloatOOBfill);
  void* fn = nullptr;
  cudaDriverEntryPointQueryResult qres;
  if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &fn, cudaEnableDefault, &qres) != cudaSuccess || !fn ||
      qres != cudaDriverEntryPointSuccess) {
    cudaGetLastError();
    return false;
  }
  constexpr int ES = (int)sizeof(R);
  cuuint32_t box[4];
  switch (order) {
    case 1: box[0] = PushBox<1, true, ES>::BX; box[1] = PushBox<1, true, ES>::BY; box[2] = PushBox<1, true, ES>::EXT; break;
    case 2: box[0] = PushBox<2, true, ES>::BX; box[1] = PushBox<2, true, ES>::BY; box[2] = PushBox<2, true, ES>::EXT; break;
    default: box[0] = PushBox<3, true, ES>::BX; box[1] = PushBox<3, true, ES>::BY; box[2] = PushBox<3, true, ES>::EXT; break;
  }
  box[3] = 6;
  if ((box[0] * es) % 16) return false;
  const cuuint64_t dims[4] = {(cuuint64_t)g.P[0], (cuuint64_t)g.P[1], (cuuint64_t)g.P[2], 6};
  const cuuint64_t strides[3] = {st1, st2, st3};
  const cuuint32_t estr[4] = {1, 1, 1, 1};
  const CUresult r = ((EncodeFn)fn)(&c.tmap_push, es == 8 ? CU_TENSOR_MAP_DATA_TYPE_FLOAT64 : CU_TENSOR_MAP_DATA_TYPE_FLOAT32, 4,
                                    (void*)g.F[0], dims, strides, box, estr, CU_TENSOR_MAP_INTERLEAVE_NONE,
                                    CU_TENSOR_MAP_SWIZZLE_NONE, CU_TENSOR_MAP_L2_PROMOTION_L2_256B,
                                    CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
  c.tma_push = r == CUDA_SUCCESS;
  return c.tma_push;
}
template bool make_push_tensor_map<double>(const Grid<double>&, int, int, int, Ctx&);
template bool make_push_tensor_map<float>(const Grid<float>&, int, int, int, Ctx&);

template <class R>
void launch_tile_kernels(const Grid<R>& g, const ParticleStep<R>& a, int order, int mode, Ctx& c) {
  switch (order) {
    case 1: launch_tile_order<R, 1>(g, a, mode, c); break;
    case 2: launch_tile_order<R, 2>(g, a, mode, c); break;
    default: launch_tile_order<R, 3>(g, a, mode, c); break;
  }
}

template void launch_tile_kernels<double>(const Grid<double>&, const ParticleStep<double>&, int, int, Ctx&);
template void launch_tile_kernels<float>(const Grid<float>&, const ParticleStep<float>&, int, int, Ctx&);

}  // namespace pic
