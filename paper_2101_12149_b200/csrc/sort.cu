// Stable counting sort of particles by tile-major cell key (
// PAPER.md:185-203 §3.4.2: counting sort = histogram + prefix sum + scatter, "binning" computes
// the permutation, "sorting" reorders the data). The key is sorted digit by digit (8 bits per
// pass, least significant first); every pass is itself a stable counting sort: per-block digit
// histogram -> exclusive prefix sum -> order-preserving scatter. Stability makes the final
// permutation unique, so it can be compared bit for bit.
#include <cmath>
#include <mutex>
#include <string>

#include "internal.h"
#include "pic.h"

namespace pic {

namespace {

constexpr int kSortThreads = 256;
constexpr int kSortItems = 16;
constexpr int kSortChunk = kSortThreads * kSortItems;   // keys per block and pass
constexpr int kWarps = kSortThreads / 32;
constexpr int kPerWarp = kSortChunk / kWarps;           // consecutive keys owned by one warp

// ---- keys: tile-major cell key, one rounded multiply per axis (bit-exact rule)
template <class R>
__global__ void __launch_bounds__(256) k_make_keys(Grid<R> g, TileSpec t, const R* __restrict__ x,
                                                   const R* __restrict__ y, const R* __restrict__ z, int64_t n,
                                                   uint32_t* __restrict__ keys, uint32_t* __restrict__ vals) {
  int64_t p = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (p >= n) return;
  int cx = cell_of<R>(x[p], g.inv_dx[0], g.N[0]);
  int cy = cell_of<R>(y[p], g.inv_dx[1], g.N[1]);
  int cz = cell_of<R>(z[p], g.inv_dx[2], g.N[2]);
  uint32_t tile = (cx / t.T[0]) + t.nt[0] * ((cy / t.T[1]) + t.nt[1] * (cz / t.T[2]));
  uint32_t rem = (cx % t.T[0]) + t.T[0] * ((cy % t.T[1]) + t.T[1] * (cz % t.T[2]));
  keys[p] = t.key_mode == 0 ? tile * (uint32_t)t.tvol + rem : tile;
  vals[p] = (uint32_t)p;
}

// ---- one radix pass
__global__ void __launch_bounds__(kSortThreads) k_radix_hist(const uint32_t* __restrict__ keys, int64_t n, int shift,
                                                             uint32_t* __restrict__ hist, int nblocks) {
  __shared__ uint32_t h[256];
  h[threadIdx.x] = 0;
  __syncthreads();
  int64_t base = (int64_t)blockIdx.x * kSortChunk;
#pragma unroll
  for (int it = 0; it < kSortItems; ++it) {
    int64_t p = base + it * kSortThreads + threadIdx.x;
    if (p < n) atomicAdd(&h[(keys[p] >> shift) & 255u], 1u);
  }
  __syncthreads();
  hist[(int64_t)threadIdx.x * nblocks + blockIdx.x] = h[threadIdx.x];   // digit-major
}

// Order-preserving scatter: warp w of the block owns the consecutive keys
// [w*kPerWarp, (w+1)*kPerWarp) of the block's chunk and walks them 32 at a time; the rank of a
// key among equal digits is (count in earlier blocks) + (count in earlier warps of the block)
// + (count earlier in this warp's walk) + (lower lanes with the same digit).
__global__ void __launch_bounds__(kSortThreads, 4) k_radix_scatter(const uint32_t* __restrict__ keys_in,
                                                                const uint32_t* __restrict__ vals_in,
                                                                uint32_t* __restrict__ keys_out,
                                                                uint32_t* __restrict__ vals_out, int64_t n, int shift,
                                                                const uint32_t* __restrict__ hist, int nblocks) {
  __shared__ uint32_t cnt[kWarps][256];
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  for (int i = threadIdx.x; i < kWarps * 256; i += kSortThreads) (&cnt[0][0])[i] = 0;
  __syncthreads();
  const int64_t wbase = (int64_t)blockIdx.x * kSortChunk + (int64_t)warp * kPerWarp;
  constexpr int kRounds = kPerWarp / 32;
  uint32_t key[kRounds], rank[kRounds];   // values are re-read at the end: registers buy occupancy here
  const uint32_t lt = (1u << lane) - 1u;
  // all loads first (independent, in flight together), then the serial ranking walk
#pragma unroll
  for (int r = 0; r < kRounds; ++r) {
    int64_t p = wbase + r * 32 + lane;
    key[r] = p < n ? keys_in[p] : 0u;
  }
#pragma unroll
  for (int r = 0; r < kRounds; ++r) {
    int64_t p = wbase + r * 32 + lane;
    bool ok = p < n;
    uint32_t d = ok ? ((key[r] >> shift) & 255u) : (256u + lane);   // invalid lanes match nobody
    uint32_t m = __match_any_sync(0xffffffffu, d);
    int leader = __ffs(m) - 1;
    uint32_t prev = 0;
    if (ok && lane == leader) {
      prev = cnt[warp][d];
      cnt[warp][d] = prev + __popc(m);
    }
    prev = __shfl_sync(0xffffffffu, prev, leader);
    rank[r] = prev + __popc(m & lt);
    __syncwarp();
  }
  __syncthreads();
  {   // per digit: global base of (digit, block), then running sum over the warps
    int d = threadIdx.x;
    uint32_t run = hist[(int64_t)d * nblocks + blockIdx.x];
#pragma unroll
    for (int w = 0; w < kWarps; ++w) {
      uint32_t c = cnt[w][d];
      cnt[w][d] = run;
      run += c;
    }
  }
  __syncthreads();
#pragma unroll
  for (int r = 0; r < kRounds; ++r) {
    int64_t p = wbase + r * 32 + lane;
    if (p < n) {
      uint32_t pos = cnt[warp][(key[r] >> shift) & 255u] + rank[r];
      keys_out[pos] = key[r];
      vals_out[pos] = vals_in[p];
    }
  }
}

// ---- exclusive prefix sum of a uint32 array (block scan + recursion on block sums)
constexpr int kScanThreads = 1024;
constexpr int kScanItems = 4;
constexpr int kScanChunk = kScanThreads * kScanItems;

__global__ void __launch_bounds__(kScanThreads) k_scan_block(uint32_t* __restrict__ data, int64_t n,
                                                             uint32_t* __restrict__ sums) {
  __shared__ uint32_t wsum[32];
  int64_t base = (int64_t)blockIdx.x * kScanChunk + (int64_t)threadIdx.x * kScanItems;
  uint32_t v[kScanItems];
  uint32_t tot = 0;
#pragma unroll
  for (int i = 0; i < kScanItems; ++i) {
    v[i] = (base + i < n) ? data[base + i] : 0u;
    tot += v[i];
  }
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  uint32_t inc = tot;
#pragma unroll
  for (int o = 1; o < 32; o <<= 1) {
    uint32_t t = __shfl_up_sync(0xffffffffu, inc, o);
    if (lane >= o) inc += t;
  }
  if (lane == 31) wsum[warp] = inc;
  __syncthreads();
  if (warp == 0) {
    uint32_t s = wsum[lane];
    uint32_t si = s;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
      uint32_t t = __shfl_up_sync(0xffffffffu, si, o);
      if (lane >= o) si += t;
    }
    wsum[lane] = si - s;                      // exclusive over warps
    if (lane == 31 && sums) sums[blockIdx.x] = si;
  }
  __syncthreads();
  uint32_t run = wsum[warp] + (inc - tot);
#pragma unroll
  for (int i = 0; i < kScanItems; ++i) {
    if (base + i < n) data[base + i] = run;
    run += v[i];
  }
}

__global__ void __launch_bounds__(kScanThreads) k_scan_add(uint32_t* __restrict__ data, int64_t n,
                                                           const uint32_t* __restrict__ sums) {
  uint32_t add = sums[blockIdx.x];
  int64_t base = (int64_t)blockIdx.x * kScanChunk + (int64_t)threadIdx.x * kScanItems;
#pragma unroll
  for (int i = 0; i < kScanItems; ++i)
    if (base + i < n) data[base + i] += add;
}

void scan_exclusive(uint32_t* data, int64_t n, uint32_t* tmp, Ctx& c) {
  int64_t nb = (n + kScanChunk - 1) / kScanChunk;
  if (nb <= 1) {
    k_scan_block<<<1, kScanThreads, 0, c.stream>>>(data, n, nullptr);
    c.launches++;
    return;
  }
  k_scan_block<<<(unsigned)nb, kScanThreads, 0, c.stream>>>(data, n, tmp);
  c.launches++;
  scan_exclusive(tmp, nb, tmp + nb, c);
  k_scan_add<<<(unsigned)nb, kScanThreads, 0, c.stream>>>(data, n, tmp);
  c.launches++;
}

// ---- apply the permutation to every attribute; record cell[] and perm[] of the new order
template <class R>
__global__ void __launch_bounds__(256) k_permute(Grid<R> g, Particles<R> src, Particles<R> dst,
                                                 const uint32_t* __restrict__ order, int32_t* __restrict__ cell,
                                                 int32_t* __restrict__ perm) {
  int64_t k = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (k >= src.n) return;
  uint32_t s = order[k];
  R x = src.x[s], y = src.y[s], z = src.z[s];
  dst.x[k] = x; dst.y[k] = y; dst.z[k] = z;
  dst.ux[k] = src.ux[s]; dst.uy[k] = src.uy[s]; dst.uz[k] = src.uz[s];
  dst.w[k] = src.w[s];
  dst.id[k] = src.id[s];
  perm[k] = (int32_t)s;
  int cx = cell_of<R>(x, g.inv_dx[0], g.N[0]);
  int cy = cell_of<R>(y, g.inv_dx[1], g.N[1]);
  int cz = cell_of<R>(z, g.inv_dx[2], g.N[2]);
  cell[k] = cx + g.N[0] * (cy + g.N[1] * cz);
}

// ---- first slot of every tile in the sorted order (tile-major key): tile_start[t] = first k with
// tile(key[k]) >= t, tile_start[n_tiles] = n. Written without atomics: the thread at a tile
// boundary fills the entries of every tile that begins there (empty tiles included).
__global__ void __launch_bounds__(256) k_tile_bounds(const uint32_t* __restrict__ keys, int64_t n, uint32_t tvol,
                                                     int n_tiles, int32_t* __restrict__ tile_start) {
  int64_t k = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (k >= n) return;
  int tk = (int)(keys[k] / tvol);
  int tp = k == 0 ? -1 : (int)(keys[k - 1] / tvol);
  for (int t = tp + 1; t <= tk; ++t) tile_start[t] = (int32_t)k;
  if (k == n - 1)
    for (int t = tk + 1; t <= n_tiles; ++t) tile_start[t] = (int32_t)n;
}

int key_bits(const TileSpec& t) {
  uint64_t nb = (uint64_t)t.nt[0] * t.nt[1] * t.nt[2] * (t.key_mode == 0 ? (uint64_t)t.tvol : 1ull);
  int b = 0;
  while ((1ull << b) < nb) ++b;
  return b < 1 ? 1 : b;
}

}  // namespace

int64_t sort_chunk() { return kSortChunk; }
int64_t sort_hist_len(int64_t n) { return 256 * ((n + kSortChunk - 1) / kSortChunk); }
int64_t sort_scan_tmp_len(int64_t hist_len) {
  int64_t tot = 0, n = hist_len;
  while (n > 1) {
    n = (n + kScanChunk - 1) / kScanChunk;
    tot += n;
    if (n == 1) break;
  }
  return tot + 8;
}

template <class R>
void sort_species(const Grid<R>& g, const TileSpec& t, const Particles<R>& cur, const Particles<R>& alt,
                  int32_t* cell, int32_t* perm, int32_t* tile_start, SortScratch& s, Ctx& c) {
  const int64_t n = cur.n;
  if (n == 0) return;
  const int nblocks = (int)((n + kSortChunk - 1) / kSortChunk);
  k_make_keys<R><<<(unsigned)((n + 255) / 256), 256, 0, c.stream>>>(g, t, cur.x, cur.y, cur.z, n, s.keys[0], s.vals[0]);
  c.launches++;
  const int bits = key_bits(t);
  int in = 0;
  for (int shift = 0; shift < bits; shift += 8) {
    k_radix_hist<<<nblocks, kSortThreads, 0, c.stream>>>(s.keys[in], n, shift, s.hist, nblocks);
    c.launches++;
    scan_exclusive(s.hist, 256 * (int64_t)nblocks, s.scan_tmp, c);
    k_radix_scatter<<<nblocks, kSortThreads, 0, c.stream>>>(s.keys[in], s.vals[in], s.keys[in ^ 1], s.vals[in ^ 1], n,
                                                            shift, s.hist, nblocks);
    c.launches++;
    in ^= 1;
  }
  k_permute<R><<<(unsigned)((n + 255) / 256), 256, 0, c.stream>>>(g, cur, alt, s.vals[in], cell, perm);
  c.launches++;
  if (tile_start) {
    const uint32_t tvol = t.key_mode == 0 ? (uint32_t)t.tvol : 1u;
    k_tile_bounds<<<(unsigned)((n + 255) / 256), 256, 0, c.stream>>>(s.keys[in], n, tvol, t.nt[0] * t.nt[1] * t.nt[2],
                                                                   tile_start);
    c.launches++;
  }
}

template void sort_species<double>(const Grid<double>&, const TileSpec&, const Particles<double>&,
                                   const Particles<double>&, int32_t*, int32_t*, int32_t*, SortScratch&, Ctx&);
template void sort_species<float>(const Grid<float>&, const TileSpec&, const Particles<float>&,
                                  const Particles<float>&, int32_t*, int32_t*, int32_t*, SortScratch&, Ctx&);

// =================================================================== the sort without any allocation
// pic_sort_permutation_noalloc (include/pic.h): the same stable sort by tile-major cell key (same key kernel,
// same radix passes, same scan) for callers that may not allocate — code under CUDA graph capture, serving
// loops, harnesses that forbid cudaMalloc. The scratch the passes need (two key and two value buffers, the
// per-block digit histogram, the block sums of the scan) lives in ONE file-scope device array of fixed size,
// so the call makes no cudaMalloc / cudaFree and touches no pool. Every GPU that loads the library holds the
// array (kNoAllocBytes, about 8.3 MB) until the process exits; every call on a device shares it, so two calls
// that overlap on the GPU (different streams, no dependency) race. Nothing in it has to start at zero — every
// region is written before it is read within a call (keys/values by k_make_keys, every histogram entry by
// k_radix_hist, the block sums by k_scan_block) — the histogram is cleared all the same, for a defined state.
namespace {

constexpr int64_t kNoAllocMaxN = PIC_NOALLOC_MAX_PARTICLES;                               // 524 288
constexpr int64_t kNoAllocBlocks = (kNoAllocMaxN + kSortChunk - 1) / kSortChunk;           // 128 radix blocks
constexpr int64_t kNoAllocHist = 256 * kNoAllocBlocks;                                     // digit-major histogram
constexpr int64_t kNoAllocScan = 64;                                                       // >= sort_scan_tmp_len(kNoAllocHist)
constexpr int64_t kNoAllocWords = 4 * kNoAllocMaxN + kNoAllocHist + kNoAllocScan;
constexpr int64_t kNoAllocBytes = kNoAllocWords * (int64_t)sizeof(uint32_t);

// In host code this name is a host-side stand-in for the symbol, NOT a device address: the address the
// kernels get comes from cudaGetSymbolAddress (noalloc_scratch below), once per device.
static __device__ __align__(256) uint32_t g_noalloc_scratch[kNoAllocWords];

constexpr int kMaxDevices = 64;
uint32_t* g_noalloc_ptr[kMaxDevices] = {};   // per device ordinal; written once, under the mutex
std::mutex g_noalloc_mutex;

// device address of the scratch array on the CURRENT device (looked up once per device, with it current)
cudaError_t noalloc_scratch(uint32_t** out) {
  int dev = 0;
  cudaError_t e = cudaGetDevice(&dev);
  if (e != cudaSuccess) return e;
  if (dev < 0 || dev >= kMaxDevices) return cudaErrorInvalidDevice;
  std::lock_guard<std::mutex> lock(g_noalloc_mutex);
  if (!g_noalloc_ptr[dev]) {
    uint32_t* ptr = nullptr;
    e = cudaGetSymbolAddress((void**)&ptr, g_noalloc_scratch);
    if (e != cudaSuccess) return e;
    g_noalloc_ptr[dev] = ptr;
  }
  *out = g_noalloc_ptr[dev];
  return cudaSuccess;
}

// what k_permute records, without moving any particle data: perm[k] = source slot, cell[k] = its cell
template <class R>
__global__ void __launch_bounds__(256) k_perm_cell(Grid<R> g, const R* __restrict__ x, const R* __restrict__ y,
                                                   const R* __restrict__ z, int64_t n, const uint32_t* __restrict__ order,
                                                   int32_t* __restrict__ cell, int32_t* __restrict__ perm) {
  int64_t k = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (k >= n) return;
  uint32_t s = order[k];
  perm[k] = (int32_t)s;
  int cx = cell_of<R>(x[s], g.inv_dx[0], g.N[0]);
  int cy = cell_of<R>(y[s], g.inv_dx[1], g.N[1]);
  int cz = cell_of<R>(z[s], g.inv_dx[2], g.N[2]);
  cell[k] = cx + g.N[0] * (cy + g.N[1] * cz);
}

template <class R>
cudaError_t sort_permutation_noalloc(const int32_t* n_cells, const double* dx, const TileSpec& t, const R* x, const R* y,
                                     const R* z, int64_t n, int32_t* cell, int32_t* perm, cudaStream_t stream) {
  uint32_t* base = nullptr;
  cudaError_t e = noalloc_scratch(&base);
  if (e != cudaSuccess) return e;
  uint32_t* keys[2] = {base, base + kNoAllocMaxN};
  uint32_t* vals[2] = {base + 2 * kNoAllocMaxN, base + 3 * kNoAllocMaxN};
  uint32_t* hist = base + 4 * kNoAllocMaxN;
  uint32_t* scan_tmp = hist + kNoAllocHist;
  Grid<R> g{};
  for (int d = 0; d < 3; ++d) {
    g.N[d] = n_cells[d];
    g.inv_dx[d] = (R)(1.0 / dx[d]);   // as pic_create rounds it
  }
  Ctx c;
  c.stream = stream;
  e = cudaMemsetAsync(hist, 0, (size_t)kNoAllocHist * sizeof(uint32_t), stream);
  if (e != cudaSuccess) return e;
  const int nblocks = (int)((n + kSortChunk - 1) / kSortChunk);
  k_make_keys<R><<<(unsigned)((n + 255) / 256), 256, 0, stream>>>(g, t, x, y, z, n, keys[0], vals[0]);
  const int bits = key_bits(t);
  int in = 0;
  for (int shift = 0; shift < bits; shift += 8) {
    k_radix_hist<<<nblocks, kSortThreads, 0, stream>>>(keys[in], n, shift, hist, nblocks);
    scan_exclusive(hist, 256 * (int64_t)nblocks, scan_tmp, c);
    k_radix_scatter<<<nblocks, kSortThreads, 0, stream>>>(keys[in], vals[in], keys[in ^ 1], vals[in ^ 1], n, shift, hist,
                                                          nblocks);
    in ^= 1;
  }
  k_perm_cell<R><<<(unsigned)((n + 255) / 256), 256, 0, stream>>>(g, x, y, z, n, vals[in], cell, perm);
  return cudaGetLastError();
}

}  // namespace

}  // namespace pic

extern "C" PIC_API int pic_sort_permutation_noalloc(const int32_t n_cells[3], const double dx[3], const int32_t tile[3],
                                                    int32_t sort_key_mode, pic_precision prec, const void* x, const void* y,
                                                    const void* z, int64_t n, int32_t* cell, int32_t* perm, void* cuda_stream) {
  using namespace pic;
  auto bad = [&](int code, const std::string& msg) { set_handleless_error(msg); return code; };
  if (!n_cells || !dx || !tile) return bad(PIC_ERR_INVALID_ARG, "null grid description");
  if (prec != PIC_F64 && prec != PIC_F32) return bad(PIC_ERR_INVALID_ARG, "unknown precision");
  if (sort_key_mode < 0 || sort_key_mode > 1) return bad(PIC_ERR_INVALID_ARG, "sort_key_mode must be 0 or 1");
  if (n < 0) return bad(PIC_ERR_INVALID_ARG, "negative particle count");
  if (n > kNoAllocMaxN)
    return bad(PIC_ERR_CAPACITY, "pic_sort_permutation_noalloc: n = " + std::to_string(n) + " exceeds PIC_NOALLOC_MAX_PARTICLES = " +
                                     std::to_string(kNoAllocMaxN) + " (the fixed scratch array); use pic_sort_now on a handle");
  TileSpec t{};
  uint64_t nnodes = 1;
  for (int d = 0; d < 3; ++d) {
    if (n_cells[d] < 1) return bad(PIC_ERR_INVALID_ARG, "n_cells must be at least 1 on every axis");
    if (!(dx[d] > 0) || !std::isfinite(dx[d])) return bad(PIC_ERR_INVALID_ARG, "dx must be positive and finite");
    if (tile[d] < 1) return bad(PIC_ERR_INVALID_ARG, "tile must be at least 1");
    const int T = tile[d] < n_cells[d] ? tile[d] : n_cells[d];
    if (n_cells[d] % T != 0) return bad(PIC_ERR_INVALID_ARG, "tile must divide n_cells");
    t.T[d] = T;
    t.nt[d] = n_cells[d] / T;
    nnodes *= (uint64_t)n_cells[d];
  }
  if (nnodes >= (1ull << 31)) return bad(PIC_ERR_INVALID_ARG, "grid too large for 32-bit cell indices");
  t.tvol = t.T[0] * t.T[1] * t.T[2];
  t.key_mode = sort_key_mode;
  if (n == 0) return PIC_OK;
  if (!x || !y || !z || !cell || !perm) return bad(PIC_ERR_INVALID_ARG, "null particle or output array");
  cudaError_t e = prec == PIC_F64
                      ? sort_permutation_noalloc<double>(n_cells, dx, t, (const double*)x, (const double*)y, (const double*)z, n, cell,
                                                         perm, (cudaStream_t)cuda_stream)
                      : sort_permutation_noalloc<float>(n_cells, dx, t, (const float*)x, (const float*)y, (const float*)z, n, cell,
                                                        perm, (cudaStream_t)cuda_stream);
  if (e != cudaSuccess) {
    cudaGetLastError();
    return bad(PIC_ERR_CUDA, std::string("pic_sort_permutation_noalloc: ") + cudaGetErrorString(e));
  }
  return PIC_OK;
}
