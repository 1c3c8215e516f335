// C ABI of libpic.so (include/pic.h): handle, memory, step orchestration. Every step of the path
// runs in the CUDA kernels of fields.cu / particles.cu / sort.cu; this file only sequences them
// on one stream.
#include "pic.h"

#include <algorithm>
#include <cmath>
#include <cstdio>
#include <cstring>
#include <map>
#include <string>
#include <utility>
#include <vector>

#include "internal.h"
#include "pool.h"

namespace pic {

static_assert(kNumPhases == PIC_NPHASE, "phase lists out of sync");

namespace {

thread_local std::string g_create_error;

__global__ void k_iota(int64_t* p, int64_t n) {
  int64_t t = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (t < n) p[t] = t;
}

// Weights of the CKC smoothed differences (include/pic.h, pic_ckc_coefficients), written in the inverse
// square spacings k_a = 1/dx_a^2 with d2 = min(dx)^2 = 1/max(k): for the difference along a, with b and c
// the transverse axes and Q = k_x k_y + k_y k_z + k_z k_x,
//   beta_ab = d2 k_b (1 - d2 k_x k_y k_z / Q) / 8,   gamma_a = d2^2 k_b k_c (1/16 - k_b k_c / (8 Q)),
//   alpha_a = 1 - 2 beta_ab - 2 beta_ac - 4 gamma_a.
// Pinned on this side by tests/test_abi.py (cubic 7/12, 1/12, 1/48; unit sum; the von Neumann bound at
// c dt = min dx; no dispersion along an axis), independently of the oracle's own copy of the scheme.
void ckc_weights(const double* dx, double* alpha, double (*beta)[3], double* gamma) {
  const double k[3] = {1.0 / (dx[0] * dx[0]), 1.0 / (dx[1] * dx[1]), 1.0 / (dx[2] * dx[2])};
  const double d2 = 1.0 / std::max(k[0], std::max(k[1], k[2]));
  const double Q = k[0] * k[1] + k[1] * k[2] + k[2] * k[0];
  const double common = (1.0 - d2 * (k[0] * k[1] * k[2]) / Q) / 8.0;
  for (int a = 0; a < 3; ++a) {
    double two_beta = 0.0, kk = 1.0;
    for (int b = 0; b < 3; ++b) {
      beta[a][b] = b == a ? 0.0 : d2 * k[b] * common;
      two_beta += 2.0 * beta[a][b];
      if (b != a) kk *= k[b];
    }
    gamma[a] = d2 * d2 * kk * (1.0 / 16.0 - kk / (8.0 * Q));
    alpha[a] = 1.0 - two_beta - 4.0 * gamma[a];
  }
}

struct SimBase {
  virtual ~SimBase() {}
  std::string err;
  int prec = 0;
  int device = 0;   // the CUDA device the handle lives on (every ABI call switches to it and back)
  virtual int add_species(int64_t n, const void* const* arr, double q, double m, pic_mem where, int32_t* id) = 0;
  virtual int set_fields(const void* const* E, const void* const* B, pic_mem where) = 0;
  virtual int step(int n) = 0;
  virtual int sync() = 0;
  virtual int get_fields(void* const* E, void* const* B, void* const* J, pic_mem where) = 0;
  virtual int get_particles(int sp, int64_t cap, void* const* out, int64_t* id, int64_t* n_out, pic_mem where) = 0;
  virtual int get_sort_state(int sp, int32_t* cell, int32_t* perm, pic_mem where) = 0;
  virtual int sort_now() = 0;
  virtual int diagnostics(double* out) = 0;
  virtual int get_rho(double* rho, pic_mem where) = 0;
  virtual int enable_timing(int on) = 0;
  virtual int phase_times(float* ms, int64_t* launches, int reset) = 0;
  virtual int64_t num_particles(int sp) const = 0;
  virtual int num_species() const = 0;
};

template <class R>
struct Species {
  Particles<R> buf[2];     // double buffer for the out-of-place sort
  int cur = 0;
  int32_t* cell = nullptr;
  int32_t* perm = nullptr;
  int32_t* tile_start = nullptr;   // n_tiles + 1 entries, valid after a sort
  bool sorted_once = false;
  double q = 0, m = 0;
};

template <class R>
struct Sim : SimBase {
  Grid<R> g{};
  TileSpec tile{};
  int order = 1;
  int sort_interval = 4;
  int deposit_mode = 0;
  bool deterministic = false;   // pic_options.deterministic: J by integer reductions (common.cuh, j_add)
  double j_bound = 0;           // no J element can exceed this in magnitude (sum over species of n max|w| |q| / (dt dA))
  double dx[3]{}, dt = 0;
  Ctx ctx;
  Pool pool;
  std::vector<Species<R>> species;
  SortScratch scratch;
  int64_t step_count = 0;
  int64_t step_launches = 0;   // kernels launched by pic_step / pic_sort_now
  // CUDA graphs (kernel-launch latency dominates once the kernels are fast): every time step
  // is captured once per "signature" (does it sort; which physical arrays hold what) and replayed as ONE
  // graph launch afterwards; the signatures of a run repeat with period 2 x sort_interval
  struct StepGraph {
    cudaGraphExec_t exec = nullptr;
    int64_t launches = 0;                    // kernels inside
    std::vector<Species<R>> after;           // host-side state the step leaves behind (buffer flips, pointer swaps)
  };
  std::map<std::vector<uint64_t>, StepGraph> graphs;
  bool use_graph = true;
  cudaStream_t cap_stream = nullptr;         // capture only (nothing ever runs on it); replays go to ctx.stream
  int64_t eager_steps = 0;                   // the first step of a handle runs eagerly (function attributes, first sort)
  unsigned long long* d_deact = nullptr;
  int* d_flags = nullptr;
  double* d_red = nullptr;   // 8 doubles of reduction scratch
  void drop_graphs() {
    for (auto& kv : graphs)
      if (kv.second.exec) cudaGraphExecDestroy(kv.second.exec);
    graphs.clear();
    eager_steps = 0;
  }
  ~Sim() override {
    cudaStreamSynchronize(ctx.stream);
    drop_graphs();
    if (cap_stream) cudaStreamDestroy(cap_stream);
    ctx.timer.destroy();
    pool.release();
    cudaGetLastError();
  }

  int fail(int code, const std::string& msg) {
    err = msg;
    return code;
  }
  int cuda_fail(cudaError_t e, const char* what) {
    cudaGetLastError();
    return fail(PIC_ERR_CUDA, std::string(what) + ": " + cudaGetErrorString(e));
  }
#define PIC_CUDA(call)                                  \
  do {                                                  \
    cudaError_t e_ = (call);                            \
    if (e_ != cudaSuccess) return cuda_fail(e_, #call); \
  } while (0)

  int check_launch(const char* what) {
    cudaError_t e = cudaGetLastError();
    if (e != cudaSuccess) return cuda_fail(e, what);
    return PIC_OK;
  }

  template <class T>
  T* palloc(size_t n) { return (T*)pool.alloc(n * sizeof(T)); }

  int init(const int32_t* n_cells, const double* dx_, double dt_, int order_, const pic_options& o) {
    order = order_;
    dt = dt_;
    sort_interval = o.sort_interval;
    deposit_mode = o.deposit_mode;
    ctx.auto_deposit = o.deposit_mode == PIC_DEPOSIT_AUTO;
    deterministic = o.deterministic != 0;
    use_graph = o.cuda_graph != 0;
    ctx.stream = (cudaStream_t)o.cuda_stream;
    PIC_CUDA(cudaGetDevice(&ctx.device));
    this->device = ctx.device;
    PIC_CUDA(cudaDeviceGetAttribute(&ctx.sm_count, cudaDevAttrMultiProcessorCount, ctx.device));
    int64_t tot = 1;
    for (int d = 0; d < 3; ++d) {
      dx[d] = dx_[d];
      g.N[d] = n_cells[d];
      g.P[d] = n_cells[d] + 2 * kGuard;
      g.periodic[d] = o.periodic[d] ? 1 : 0;
      g.inv_dx[d] = (R)(1.0 / dx_[d]);
      g.L[d] = (R)(n_cells[d] * dx_[d]);
      g.cB[d] = (R)(dt_ / (2.0 * dx_[d]));
      g.cE[d] = (R)(kC * kC * dt_ / dx_[d]);
      tot *= g.P[d];
      int T = o.tile[d] < n_cells[d] ? o.tile[d] : n_cells[d];
      tile.T[d] = T;
      tile.nt[d] = n_cells[d] / T;
    }
    if (tot >= ((int64_t)1 << 31)) return fail(PIC_ERR_INVALID_ARG, "grid too large for 32-bit field indices");
    tile.tvol = tile.T[0] * tile.T[1] * tile.T[2];
    tile.key_mode = o.sort_key_mode;
    uint64_t nbins = (uint64_t)tile.nt[0] * tile.nt[1] * tile.nt[2] * (tile.key_mode == 0 ? (uint64_t)tile.tvol : 1ull);
    if (nbins > 0xffffffffull) return fail(PIC_ERR_INVALID_ARG, "too many sort bins for a 32-bit key");
    g.sy = g.P[0];
    g.sz = g.P[0] * g.P[1];
    g.org = kGuard + g.sy * kGuard + g.sz * kGuard;
    g.cJ = (R)(dt_ / kEps0);
    g.inv_c2 = (R)(1.0 / (kC * kC));
    g.dt = (R)dt_;
    g.pusher = o.pusher;
    g.gather_mode = o.gather_mode;
    g.solver = o.solver;
    {
      double al[3], be[3][3], ga[3];
      ckc_weights(dx_, al, be, ga);
      for (int a = 0; a < 3; ++a) {
        g.ck_a[a] = (R)al[a];
        g.ck_g[a] = (R)ga[a];
        for (int b = 0; b < 3; ++b) g.ck_b[a][b] = (R)be[a][b];
      }
    }
    // one allocation for the nine field arrays
    R* base = palloc<R>((size_t)tot * 9);
    if (!base) return fail(PIC_ERR_OOM, "field allocation failed");
    for (int c = 0; c < 6; ++c) g.F[c] = base + (size_t)tot * c;
    for (int c = 0; c < 3; ++c) g.J[c] = base + (size_t)tot * (6 + c);
    PIC_CUDA(cudaMemsetAsync(base, 0, (size_t)tot * 9 * sizeof(R), ctx.stream));
    make_push_tensor_map<R>(g, order, tile.T[0], o.box_staging, ctx);
    g.Jfix[0] = g.Jfix[1] = nullptr;
    g.fix_scale[0] = g.fix_scale[1] = g.fix_inv[0] = g.fix_inv[1] = 0.0;
    if (deterministic) {
      long long* fx = palloc<long long>((size_t)tot * 6);
      if (!fx) return fail(PIC_ERR_OOM, "fixed-point J allocation failed");
      g.Jfix[0] = fx;
      g.Jfix[1] = fx + (size_t)tot * 3;
    }
    d_deact = palloc<unsigned long long>(1);
    d_flags = palloc<int>(2);
    d_red = palloc<double>(8);
    if (!d_deact || !d_flags || !d_red) return fail(PIC_ERR_OOM, "scratch allocation failed");
    PIC_CUDA(cudaMemsetAsync(d_deact, 0, sizeof(unsigned long long), ctx.stream));
    PIC_CUDA(cudaStreamSynchronize(ctx.stream));
    if (use_graph && cudaStreamCreateWithFlags(&cap_stream, cudaStreamNonBlocking) != cudaSuccess) {
      cudaGetLastError();
      cap_stream = nullptr;
      use_graph = false;
    }
    return PIC_OK;
  }

  int copy_in(void* dst, const void* src, size_t bytes, pic_mem where) {
    PIC_CUDA(cudaMemcpyAsync(dst, src, bytes, where == PIC_HOST ? cudaMemcpyHostToDevice : cudaMemcpyDeviceToDevice, ctx.stream));
    return PIC_OK;
  }
  int copy_out(void* dst, const void* src, size_t bytes, pic_mem where) {
    PIC_CUDA(cudaMemcpyAsync(dst, src, bytes, where == PIC_HOST ? cudaMemcpyDeviceToHost : cudaMemcpyDeviceToDevice, ctx.stream));
    return PIC_OK;
  }

  int read_flags(int* f) {
    PIC_CUDA(cudaMemcpyAsync(f, d_flags, 2 * sizeof(int), cudaMemcpyDeviceToHost, ctx.stream));
    PIC_CUDA(cudaStreamSynchronize(ctx.stream));
    return PIC_OK;
  }

  void free_particles(Particles<R>& p) {
    R** a[7] = {&p.x, &p.y, &p.z, &p.ux, &p.uy, &p.uz, &p.w};
    for (auto q : a) { pool.free(*q); *q = nullptr; }
    pool.free(p.id);
    p.id = nullptr;
  }
  bool alloc_particles(Particles<R>& p, int64_t n) {
    R** a[7] = {&p.x, &p.y, &p.z, &p.ux, &p.uy, &p.uz, &p.w};
    size_t cnt = (size_t)(n > 0 ? n : 1);
    for (auto q : a) {
      *q = palloc<R>(cnt);
      if (!*q) return false;
    }
    p.id = palloc<int64_t>(cnt);
    p.n = n;
    return p.id != nullptr;
  }

  int ensure_scratch(int64_t n) {
    if (n <= scratch.cap) return PIC_OK;
    for (int i = 0; i < 2; ++i) { pool.free(scratch.keys[i]); pool.free(scratch.vals[i]); }
    pool.free(scratch.hist);
    pool.free(scratch.scan_tmp);
    pool.free(scratch.stray_list);
    pool.free(scratch.stray_count);
    scratch = SortScratch();
    scratch.hist_len = sort_hist_len(n);
    scratch.scan_len = sort_scan_tmp_len(scratch.hist_len);
    for (int i = 0; i < 2; ++i) {
      scratch.keys[i] = palloc<uint32_t>((size_t)n);
      scratch.vals[i] = palloc<uint32_t>((size_t)n);
      if (!scratch.keys[i] || !scratch.vals[i]) return fail(PIC_ERR_OOM, "sort scratch allocation failed");
    }
    scratch.hist = palloc<uint32_t>((size_t)scratch.hist_len);
    scratch.scan_tmp = palloc<uint32_t>((size_t)scratch.scan_len);
    scratch.stray_list = palloc<int32_t>((size_t)n);
    scratch.stray_count = palloc<unsigned int>(1);
    if (!scratch.hist || !scratch.scan_tmp || !scratch.stray_list || !scratch.stray_count)
      return fail(PIC_ERR_OOM, "sort scratch allocation failed");
    scratch.cap = n;
    return PIC_OK;
  }

  int add_species(int64_t n, const void* const* arr, double q, double m, pic_mem where, int32_t* id) override {
    if (n < 0 || !(m > 0) || !std::isfinite(q) || !std::isfinite(m)) return fail(PIC_ERR_INVALID_ARG, "bad n, charge or mass");
    if (n >= ((int64_t)1 << 31)) return fail(PIC_ERR_INVALID_ARG, "more than 2^31-1 particles in one species");
    for (int a = 0; a < 7; ++a)
      if (n > 0 && !arr[a]) return fail(PIC_ERR_INVALID_ARG, "null particle array");
    drop_graphs();   // the species list and the scratch buffers are part of every captured step
    Species<R> sp;
    sp.q = q;
    sp.m = m;
    {   // everything this species needs, in one chunk: two buffer sets, cell, perm, tile starts, sort scratch
      const size_t slack = 512;   // the pool's alignment, per array
      const size_t nn = (size_t)(n > 0 ? n : 1);
      size_t need = 2 * (7 * (nn * sizeof(R) + slack) + nn * sizeof(int64_t) + slack) + 2 * (nn * sizeof(int32_t) + slack) +
                    ((size_t)tile.nt[0] * tile.nt[1] * tile.nt[2] + 1) * sizeof(int32_t) + slack;
      if (n > scratch.cap)
        need += 5 * (nn * sizeof(uint32_t) + slack) + ((size_t)sort_hist_len(n) + (size_t)sort_scan_tmp_len(sort_hist_len(n))) * sizeof(uint32_t) +
                3 * slack;
      pool.reserve(need);
    }
    bool ok = alloc_particles(sp.buf[0], n) && alloc_particles(sp.buf[1], n);
    sp.cell = palloc<int32_t>((size_t)(n > 0 ? n : 1));
    sp.perm = palloc<int32_t>((size_t)(n > 0 ? n : 1));
    sp.tile_start = palloc<int32_t>((size_t)tile.nt[0] * tile.nt[1] * tile.nt[2] + 1);
    auto cleanup = [&]() {
      free_particles(sp.buf[0]); free_particles(sp.buf[1]);
      pool.free(sp.cell); pool.free(sp.perm); pool.free(sp.tile_start);
    };
    if (!ok || !sp.cell || !sp.perm || !sp.tile_start) { cleanup(); return fail(PIC_ERR_OOM, "particle allocation failed"); }
    for (int b = 0; b < 2; ++b) {
      sp.buf[b].kq = (R)(q * dt / (2.0 * m));
      sp.buf[b].jf[0] = (R)(q / (dt * dx[1] * dx[2]));
      sp.buf[b].jf[1] = (R)(q / (dt * dx[0] * dx[2]));
      sp.buf[b].jf[2] = (R)(q / (dt * dx[0] * dx[1]));
    }
    Particles<R>& p = sp.buf[0];
    R* dst[7] = {p.x, p.y, p.z, p.ux, p.uy, p.uz, p.w};
    for (int a = 0; a < 7 && n > 0; ++a) {
      int rc = copy_in(dst[a], arr[a], (size_t)n * sizeof(R), where);
      if (rc) { cleanup(); return rc; }
    }
    if (n > 0) {
      k_iota<<<(unsigned)((n + 255) / 256), 256, 0, ctx.stream>>>(p.id, n);
      ctx.launches++;
    }
    cudaMemsetAsync(d_flags, 0, 2 * sizeof(int), ctx.stream);
    launch_validate_particles<R>(g, p, d_flags, ctx);
    int f[2] = {0, 0};
    int rc = read_flags(f);
    if (rc == PIC_OK) rc = check_launch("add_species kernels");
    if (rc) { cleanup(); return rc; }
    if (f[0]) { cleanup(); return fail(PIC_ERR_INVALID_ARG, "non-finite particle value"); }
    if (f[1]) { cleanup(); return fail(PIC_ERR_OUT_OF_DOMAIN, "particle position outside [0, L)"); }
    rc = ensure_scratch(n);
    if (rc) { cleanup(); return rc; }
    if (deterministic && n > 0) {
      // every contribution of a particle to a J element is at most |q| w / (dt dA) in magnitude (the prefix of
      // the Esirkepov weights is a difference of shape products), so n max|w| |q| / (dt min dA) bounds any sum;
      // max is exact and order-free, so the scale below is the same in every run
      double wmax = 0.0;
      cudaMemsetAsync(d_red, 0, sizeof(double), ctx.stream);
      launch_max_abs<R>(p.w, n, d_red, ctx);
      PIC_CUDA(cudaMemcpyAsync(&wmax, d_red, sizeof(double), cudaMemcpyDeviceToHost, ctx.stream));
      PIC_CUDA(cudaStreamSynchronize(ctx.stream));
      const double dA = std::min(dx[0] * dx[1], std::min(dx[1] * dx[2], dx[0] * dx[2]));
      j_bound += (double)n * wmax * std::fabs(q) / (dt * dA);
      if (j_bound > 0) {
        int e = 0;
        std::frexp(j_bound, &e);                       // j_bound < 2^e
        g.fix_scale[0] = std::ldexp(1.0, 61 - e);      // |sum| 2^(61-e) < 2^61: no overflow, whatever arrives
        g.fix_scale[1] = std::ldexp(1.0, 61 - e + 40); // the low part: 40 more bits, |lo| <= 2^39 per contribution
        g.fix_inv[0] = 1.0 / g.fix_scale[0];
        g.fix_inv[1] = 1.0 / g.fix_scale[1];
      }
    }
    species.push_back(sp);
    if (id) *id = (int32_t)species.size() - 1;
    return PIC_OK;
  }

  int set_fields(const void* const* E, const void* const* B, pic_mem where) override {
    if (!E || !B) return fail(PIC_ERR_INVALID_ARG, "null field pointer array");
    for (int c = 0; c < 3; ++c)
      if (!E[c] || !B[c]) return fail(PIC_ERR_INVALID_ARG, "null field array");
    size_t nv = (size_t)g.N[0] * g.N[1] * g.N[2];
    R* stage = nullptr;
    if (where == PIC_HOST) {
      stage = palloc<R>(nv);
      if (!stage) return fail(PIC_ERR_OOM, "staging allocation failed");
    }
    cudaMemsetAsync(d_flags, 0, 2 * sizeof(int), ctx.stream);
    // validate everything before overwriting anything
    for (int c = 0; c < 6; ++c) {
      const R* src = (const R*)(c < 3 ? E[c] : B[c - 3]);
      if (where == PIC_HOST) {
        int rc = copy_in(stage, src, nv * sizeof(R), where);
        if (rc) { pool.free(stage); return rc; }
        src = stage;
      }
      launch_validate_array<R>(src, (int64_t)nv, d_flags, ctx);
    }
    int f[2] = {0, 0};
    int rc = read_flags(f);
    if (rc) { pool.free(stage); return rc; }
    if (f[0]) { pool.free(stage); return fail(PIC_ERR_INVALID_ARG, "non-finite field value"); }
    for (int c = 0; c < 6; ++c) {
      const R* src = (const R*)(c < 3 ? E[c] : B[c - 3]);
      if (where == PIC_HOST) {
        rc = copy_in(stage, src, nv * sizeof(R), where);
        if (rc) { pool.free(stage); return rc; }
        src = stage;
      }
      cudaMemsetAsync(g.F[c], 0, (size_t)g.padded_total() * sizeof(R), ctx.stream);
      launch_pack<R>(g, src, g.F[c], ctx);
    }
    launch_fill_guards<R>(g, g.F, 6, ctx);
    pool.free(stage);
    PIC_CUDA(cudaStreamSynchronize(ctx.stream));
    return check_launch("set_fields kernels");
  }

  void do_sort() {
    for (auto& sp : species) {
      if (sp.buf[sp.cur].n == 0) { sp.sorted_once = true; continue; }
      sort_species<R>(g, tile, sp.buf[sp.cur], sp.buf[sp.cur ^ 1], sp.cell, sp.perm, sp.tile_start, scratch, ctx);
      sp.cur ^= 1;
      sp.sorted_once = true;
    }
  }

  // AUTO: the tile kernels need the cell-sorted order, bins of at most 8 cells per axis and (unless asked
  // for) enough cells per tile to pay for a CTA; until the first sort the fused per-particle kernel runs
  int pick_mode(const Species<R>& sp) const {
    const bool tiles_ok = sp.sorted_once && tile.T[0] <= 8 && tile.T[1] <= 8 && tile.T[2] <= 8 &&
                          (deposit_mode != PIC_DEPOSIT_AUTO || tile.T[0] * tile.T[1] * tile.T[2] >= 64);
    const bool want_tile = deposit_mode == PIC_DEPOSIT_TILE || deposit_mode == PIC_DEPOSIT_TILE_MMA ||
                           deposit_mode == PIC_DEPOSIT_FUSED;
    if (want_tile && !tiles_ok) return sp.sorted_once ? kDepositCoop : kDepositGlobal;
    // fp32 has no fused kernel (its contraction is the fp64 tensor pipe's): the split tile kernels
    if (deposit_mode == PIC_DEPOSIT_FUSED && sizeof(R) == 4) return kDepositTile;
    if (deposit_mode != PIC_DEPOSIT_AUTO) return deposit_mode;
    // fp64: push, then the tensor-pipe deposition (the one-kernel form, PIC_DEPOSIT_FUSED, measured 9 % slower:
    // DESIGN.md section 6); fp32: push, then the lane-group deposition (its sums run on the fp32 pipe)
    const int tile_mode = sizeof(R) == 8 ? kDepositTileMma : kDepositTile;
    return tiles_ok ? tile_mode : (sp.sorted_once ? kDepositCoop : kDepositGlobal);
  }
  void particle_step(Species<R>& sp) {
    ParticleStep<R> a;
    a.cur = sp.buf[sp.cur];
    a.alt = sp.buf[sp.cur ^ 1];
    a.cell_sorted = sp.sorted_once ? sp.cell : nullptr;
    a.tile_start = sp.tile_start;
    a.tiles = tile;
    a.stray_list = scratch.stray_list;
    a.stray_count = scratch.stray_count;
    a.deactivated = d_deact;
    if (launch_particles<R>(g, a, order, pick_mode(sp), ctx)) {
      Particles<R>&c0 = sp.buf[sp.cur], &c1 = sp.buf[sp.cur ^ 1];
      std::swap(c0.x, c1.x);
      std::swap(c0.y, c1.y);
      std::swap(c0.z, c1.z);
    }
  }

  struct StepBounds { int loB[3], hiB[3], loE[3], hiE[3], lo0[3], hi0[3]; };
  StepBounds step_bounds() const {
    StepBounds b;
    for (int d = 0; d < 3; ++d) {
      b.lo0[d] = 0; b.hi0[d] = g.N[d];
      // Yee: the second B half-step reads E one layer up; CKC also reads one layer to every side, so its
      // E update is widened to [-1, N+2) and its first B half-step to [-2, N+2) (guards are 4 deep)
      const int wide = g.solver == PIC_SOLVER_CKC ? 2 : 1;
      b.loB[d] = g.periodic[d] ? -wide : 0;
      b.hiB[d] = g.periodic[d] ? g.N[d] + wide : g.N[d];
      b.loE[d] = g.periodic[d] ? -(wide - 1) : 0;
      b.hiE[d] = b.hiB[d];
    }
    return b;
  }

  // one time step: issues every launch on ctx.stream and advances the host-side state
  void step_body(const StepBounds& b) {
    const size_t jbytes = (size_t)g.padded_total() * 3 * sizeof(R);
    if (sort_interval > 0 && step_count % sort_interval == 0) {
      ScopedPhase ph(ctx, kPhaseSort);
      do_sort();
    }
    {
      ScopedPhase ph(ctx, kPhaseFields);
      cudaMemsetAsync(g.J[0], 0, jbytes, ctx.stream);   // the three J arrays are contiguous
      if (deterministic) cudaMemsetAsync(g.Jfix[0], 0, (size_t)g.padded_total() * 6 * sizeof(long long), ctx.stream);
    }
    for (auto& sp : species) particle_step(sp);         // timed per kernel in particles.cu
    {
      ScopedPhase ph(ctx, kPhaseFields);
      if (deterministic && g.fix_scale[0] != 0.0) launch_fix_to_J<R>(g, ctx);   // integer sums -> J
      launch_fold_J<R>(g, ctx);                    // SumBoundary
      launch_fill_guards<R>(g, g.J, 3, ctx);       // J images for the widened E update
      launch_push_B<R>(g, b.loB, b.hiB, ctx);      // widened by one layer on periodic axes, so
      launch_push_E<R>(g, b.loE, b.hiE, ctx);      // the valid region never reads a stale guard
      launch_push_B<R>(g, b.lo0, b.hi0, ctx);
      launch_fill_guards<R>(g, g.F, 6, ctx);       // FillBoundary
    }
    step_count++;
  }

  // what a captured step depends on besides the (fixed) grid: does it sort, and which arrays play which role
  std::vector<uint64_t> signature() const {
    std::vector<uint64_t> v;
    v.push_back(sort_interval > 0 && step_count % sort_interval == 0);
    for (const auto& sp : species) {
      v.push_back((uint64_t)sp.cur | ((uint64_t)sp.sorted_once << 1));
      for (int b = 0; b < 2; ++b) {
        v.push_back((uint64_t)(uintptr_t)sp.buf[b].x);
        v.push_back((uint64_t)(uintptr_t)sp.buf[b].y);
        v.push_back((uint64_t)(uintptr_t)sp.buf[b].z);
      }
    }
    return v;
  }

  int step(int n) override {
    if (n < 0) return fail(PIC_ERR_INVALID_ARG, "negative step count");
    const StepBounds b = step_bounds();
    const int64_t launches0 = ctx.launches;
    for (int s = 0; s < n; ++s) {
      // eager: per-kernel timing is on, graphs are off, or this is the handle's first step
      if (!use_graph || ctx.timer.on || eager_steps < 1) {
        step_body(b);
        eager_steps++;
        if (ctx.timer.spans.size() > 3000) ctx.timer.fold_completed();   // never waits: pic_step stays asynchronous
        continue;
      }
      const std::vector<uint64_t> sig = signature();
      auto it = graphs.find(sig);
      if (it == graphs.end()) {
        const int64_t l0 = ctx.launches;
        cudaStream_t user = ctx.stream;
        if (cudaStreamBeginCapture(cap_stream, cudaStreamCaptureModeThreadLocal) != cudaSuccess) {
          cudaGetLastError();
          use_graph = false;
          step_body(b);
          continue;
        }
        ctx.stream = cap_stream;
        step_body(b);                              // recorded, not run; the host-side state moves on
        ctx.stream = user;
        cudaGraph_t gr = nullptr;
        StepGraph sg;
        cudaError_t e = cudaStreamEndCapture(cap_stream, &gr);
        if (e == cudaSuccess) e = cudaGraphInstantiate(&sg.exec, gr, 0);
        if (gr) cudaGraphDestroy(gr);
        if (e != cudaSuccess) return cuda_fail(e, "CUDA graph capture of a time step");
        sg.launches = ctx.launches - l0;
        ctx.launches = l0;
        sg.after = species;
        it = graphs.emplace(sig, std::move(sg)).first;
      } else {
        species = it->second.after;
        step_count++;
      }
      cudaError_t e = cudaGraphLaunch(it->second.exec, ctx.stream);
      if (e != cudaSuccess) return cuda_fail(e, "cudaGraphLaunch");
      ctx.launches += it->second.launches;
    }
    step_launches += ctx.launches - launches0;
    return check_launch("pic_step launch");
  }

  int sync() override {
    PIC_CUDA(cudaStreamSynchronize(ctx.stream));
    return check_launch("asynchronous kernel fault");
  }

  int get_fields(void* const* E, void* const* B, void* const* J, pic_mem where) override {
    size_t nv = (size_t)g.N[0] * g.N[1] * g.N[2];
    R* stage = nullptr;
    if (where == PIC_HOST) {
      stage = palloc<R>(nv);
      if (!stage) return fail(PIC_ERR_OOM, "staging allocation failed");
    }
    void* const* grp[3] = {E, B, J};
    for (int gi = 0; gi < 3; ++gi) {
      if (!grp[gi]) continue;
      for (int c = 0; c < 3; ++c) {
        if (!grp[gi][c]) { pool.free(stage); return fail(PIC_ERR_INVALID_ARG, "null field array"); }
        const R* src = gi == 0 ? g.F[c] : gi == 1 ? g.F[3 + c] : g.J[c];
        if (where == PIC_HOST) {
          launch_unpack<R>(g, src, stage, ctx);
          int rc = copy_out(grp[gi][c], stage, nv * sizeof(R), where);
          if (rc) { pool.free(stage); return rc; }
        } else {
          launch_unpack<R>(g, src, (R*)grp[gi][c], ctx);
        }
      }
    }
    pool.free(stage);
    return sync();
  }

  int get_particles(int isp, int64_t cap, void* const* out, int64_t* id, int64_t* n_out, pic_mem where) override {
    if (isp < 0 || isp >= (int)species.size()) return fail(PIC_ERR_INVALID_ARG, "no such species");
    Particles<R>& p = species[isp].buf[species[isp].cur];
    if (n_out) *n_out = p.n;
    if (cap < p.n) return fail(PIC_ERR_CAPACITY, "output capacity below particle count");
    R* src[7] = {p.x, p.y, p.z, p.ux, p.uy, p.uz, p.w};
    for (int a = 0; a < 7; ++a)
      if (out[a] && p.n > 0) {
        int rc = copy_out(out[a], src[a], (size_t)p.n * sizeof(R), where);
        if (rc) return rc;
      }
    if (id && p.n > 0) {
      int rc = copy_out(id, p.id, (size_t)p.n * sizeof(int64_t), where);
      if (rc) return rc;
    }
    return sync();
  }

  int get_sort_state(int isp, int32_t* cell, int32_t* perm, pic_mem where) override {
    if (isp < 0 || isp >= (int)species.size()) return fail(PIC_ERR_INVALID_ARG, "no such species");
    Species<R>& sp = species[isp];
    if (!sp.sorted_once) return fail(PIC_ERR_INVALID_ARG, "species has not been sorted yet");
    int64_t n = sp.buf[sp.cur].n;
    if (cell && n > 0) { int rc = copy_out(cell, sp.cell, (size_t)n * 4, where); if (rc) return rc; }
    if (perm && n > 0) { int rc = copy_out(perm, sp.perm, (size_t)n * 4, where); if (rc) return rc; }
    return sync();
  }

  int sort_now() override {
    const int64_t launches0 = ctx.launches;
    {
      ScopedPhase ph(ctx, kPhaseSort);
      do_sort();
    }
    step_launches += ctx.launches - launches0;
    return check_launch("sort launch");
  }

  int fill_rho(double* rho) {
    size_t nv = (size_t)g.N[0] * g.N[1] * g.N[2];
    PIC_CUDA(cudaMemsetAsync(rho, 0, nv * sizeof(double), ctx.stream));
    for (auto& sp : species) launch_rho<R>(g, sp.buf[sp.cur], order, sp.q, rho, ctx);
    return PIC_OK;
  }

  int diagnostics(double* out) override {
    if (!out) return fail(PIC_ERR_INVALID_ARG, "null output");
    size_t nv = (size_t)g.N[0] * g.N[1] * g.N[2];
    double* rho = palloc<double>(nv);
    if (!rho) return fail(PIC_ERR_OOM, "rho allocation failed");
    double h[8];
    unsigned long long deact = 0;
    // the pool block goes back on every path (stream order makes an immediate free safe)
    int rc = [&]() -> int {
      PIC_CUDA(cudaMemsetAsync(d_red, 0, 8 * sizeof(double), ctx.stream));
      launch_field_energy<R>(g, d_red, ctx);
      for (auto& sp : species) launch_particle_sums<R>(sp.buf[sp.cur], sp.q, sp.m, d_red + 2, ctx);
      int r = fill_rho(rho);
      if (r) return r;
      launch_gauss<R>(g, rho, d_red + 4, ctx);
      PIC_CUDA(cudaMemcpyAsync(h, d_red, sizeof(h), cudaMemcpyDeviceToHost, ctx.stream));
      PIC_CUDA(cudaMemcpyAsync(&deact, d_deact, sizeof(deact), cudaMemcpyDeviceToHost, ctx.stream));
      return sync();
    }();
    pool.free(rho);
    if (rc) return rc;
    double dv = dx[0] * dx[1] * dx[2];
    out[PIC_DIAG_FIELD_E] = 0.5 * kEps0 * h[0] * dv;
    out[PIC_DIAG_FIELD_B] = 0.5 * kEps0 * kC * kC * h[1] * dv;
    out[PIC_DIAG_KINETIC] = h[2];
    out[PIC_DIAG_CHARGE] = h[3];
    out[PIC_DIAG_GAUSS_MAX] = h[4];
    out[PIC_DIAG_RHO_MAX] = h[5];
    out[PIC_DIAG_DEACTIVATED] = (double)deact;
    out[PIC_DIAG_STEPS] = (double)step_count;
    out[PIC_DIAG_POOL_CHUNKS] = (double)pool.n_chunks();
    out[PIC_DIAG_POOL_BYTES] = (double)pool.bytes_held();
    out[PIC_DIAG_LAUNCHES] = (double)ctx.launches;
    out[PIC_DIAG_STEP_LAUNCHES] = (double)step_launches;
    return PIC_OK;
  }

  int get_rho(double* rho, pic_mem where) override {
    if (!rho) return fail(PIC_ERR_INVALID_ARG, "null output");
    size_t nv = (size_t)g.N[0] * g.N[1] * g.N[2];
    double* d = where == PIC_DEVICE ? rho : palloc<double>(nv);
    if (!d) return fail(PIC_ERR_OOM, "rho allocation failed");
    int rc = fill_rho(d);
    if (rc == PIC_OK && where == PIC_HOST) rc = copy_out(rho, d, nv * sizeof(double), where);
    if (where == PIC_HOST) pool.free(d);
    if (rc) return rc;
    return sync();
  }

  int enable_timing(int on) override {
    if (!on && ctx.timer.on) ctx.timer.fold();
    ctx.timer.on = on != 0;
    return PIC_OK;
  }
  int phase_times(float* ms, int64_t* launches, int reset) override {
    if (!ms) return fail(PIC_ERR_INVALID_ARG, "null output");
    ctx.timer.fold();
    for (int i = 0; i < PIC_NPHASE; ++i) {
      ms[i] = ctx.timer.ms[i];
      if (launches) launches[i] = ctx.timer.count[i];
    }
    if (reset) ctx.timer.reset();
    return PIC_OK;
  }

  int64_t num_particles(int isp) const override {
    if (isp < 0 || isp >= (int)species.size()) return -1;
    return species[isp].buf[species[isp].cur].n;
  }
  int num_species() const override { return (int)species.size(); }
#undef PIC_CUDA
};

}  // namespace

// for entry points outside this file that have no handle: the text pic_last_error(NULL) returns (this thread)
void set_handleless_error(const std::string& msg) { g_create_error = msg; }

}  // namespace pic

struct pic_sim {
  pic::SimBase* impl;
};

extern "C" {

void pic_default_options(pic_options* o) {
  if (!o) return;
  std::memset(o, 0, sizeof(*o));
  for (int d = 0; d < 3; ++d) { o->periodic[d] = 1; o->tile[d] = 8; }
  o->sort_interval = 4;
  o->sort_key_mode = 0;
  o->deposit_mode = PIC_DEPOSIT_AUTO;
  o->pusher = PIC_PUSHER_BORIS;
  o->gather_mode = PIC_GATHER_UNIFORM;
  o->solver = PIC_SOLVER_YEE;
  o->deterministic = 0;
  o->cuda_graph = 1;
  o->box_staging = PIC_STAGE_AUTO;
  o->cuda_stream = nullptr;
}

int pic_create(const int32_t n_cells[3], const double dx[3], double dt, int shape_order, pic_precision prec,
               const pic_options* opt, pic_sim** out) {
  using namespace pic;
  auto bad = [&](int code, const char* msg) { g_create_error = msg; return code; };
  if (!out) return bad(PIC_ERR_INVALID_ARG, "out is NULL");
  *out = nullptr;
  if (!n_cells || !dx) return bad(PIC_ERR_INVALID_ARG, "n_cells or dx is NULL");
  pic_options o;
  pic_default_options(&o);
  if (opt) o = *opt;
  if (shape_order < 1 || shape_order > 3) return bad(PIC_ERR_INVALID_ARG, "shape_order must be 1, 2 or 3");
  if (prec != PIC_F64 && prec != PIC_F32) return bad(PIC_ERR_INVALID_ARG, "unknown precision");
  if (o.sort_interval < 0 || o.sort_key_mode < 0 || o.sort_key_mode > 1 || o.deposit_mode < 0 ||
      o.deposit_mode > 5 || o.pusher < 0 || o.pusher > 1 || o.gather_mode < 0 || o.gather_mode > 1 ||
      o.solver < 0 || o.solver > 1 || o.deterministic < 0 || o.deterministic > 1 ||
      o.cuda_graph < 0 || o.cuda_graph > 1 || o.box_staging < 0 || o.box_staging > 2)
    return bad(PIC_ERR_INVALID_ARG, "bad option value");
  double s2 = 0;
  for (int d = 0; d < 3; ++d) {
    if (n_cells[d] < kGuard) return bad(PIC_ERR_INVALID_ARG, "n_cells must be at least 4 on every axis");
    if (!(dx[d] > 0) || !std::isfinite(dx[d])) return bad(PIC_ERR_INVALID_ARG, "dx must be positive and finite");
    if (o.tile[d] < 1) return bad(PIC_ERR_INVALID_ARG, "tile must be at least 1");
    int T = o.tile[d] < n_cells[d] ? o.tile[d] : n_cells[d];
    if (n_cells[d] % T != 0) return bad(PIC_ERR_INVALID_ARG, "tile must divide n_cells");
    s2 += 1.0 / (dx[d] * dx[d]);
  }
  if (!(dt > 0) || !std::isfinite(dt)) return bad(PIC_ERR_INVALID_ARG, "dt must be positive and finite");
  if (o.solver == PIC_SOLVER_YEE && dt * kC * std::sqrt(s2) > 1.0)
    return bad(PIC_ERR_CFL, "dt violates the CFL limit dt*c*sqrt(sum 1/dx^2) <= 1");
  if (o.solver == PIC_SOLVER_CKC && dt * kC > std::min(dx[0], std::min(dx[1], dx[2])) * (1.0 + 1e-12))
    return bad(PIC_ERR_CFL, "dt violates the CKC limit c*dt <= min(dx)");
  int ndev = 0;
  cudaError_t e = cudaGetDeviceCount(&ndev);
  if (e != cudaSuccess || ndev == 0) {
    cudaGetLastError();
    return bad(PIC_ERR_CUDA, "no usable CUDA device (this library has no CPU fallback)");
  }
  SimBase* impl = nullptr;
  int rc;
  if (prec == PIC_F64) {
    auto* s = new Sim<double>();
    rc = s->init(n_cells, dx, dt, shape_order, o);
    impl = s;
  } else {
    auto* s = new Sim<float>();
    rc = s->init(n_cells, dx, dt, shape_order, o);
    impl = s;
  }
  impl->prec = (int)prec;
  if (rc != PIC_OK) {
    g_create_error = impl->err;
    delete impl;
    return rc;
  }
  *out = new pic_sim{impl};
  g_create_error.clear();
  return PIC_OK;
}

// A handle belongs to the device that was current at pic_create: its memory, stream, function attributes
// and tensor map live there. Every call on a handle makes that device current for its duration and restores
// the caller's afterwards, so a process that drives several GPUs can hold one handle per device.
struct DeviceGuard {
  int prev = -1;
  bool switched = false;
  explicit DeviceGuard(int dev) {
    if (cudaGetDevice(&prev) == cudaSuccess && prev != dev) switched = cudaSetDevice(dev) == cudaSuccess;
  }
  ~DeviceGuard() {
    if (switched) cudaSetDevice(prev);
  }
};
#define SIM_OR_FAIL(s)                               \
  if (!(s) || !(s)->impl) return PIC_ERR_INVALID_ARG; \
  DeviceGuard device_guard_((s)->impl->device)

int pic_add_species(pic_sim* sim, int64_t n, const void* x, const void* y, const void* z, const void* ux,
                    const void* uy, const void* uz, const void* w, double charge, double mass, pic_mem where,
                    int32_t* species_id) {
  SIM_OR_FAIL(sim);
  const void* arr[7] = {x, y, z, ux, uy, uz, w};
  return sim->impl->add_species(n, arr, charge, mass, where, species_id);
}

int pic_set_fields(pic_sim* sim, const void* const E[3], const void* const B[3], pic_mem where) {
  SIM_OR_FAIL(sim);
  return sim->impl->set_fields(E, B, where);
}

int pic_step(pic_sim* sim, int32_t n) {
  SIM_OR_FAIL(sim);
  return sim->impl->step(n);
}

int pic_synchronize(pic_sim* sim) {
  SIM_OR_FAIL(sim);
  return sim->impl->sync();
}

int pic_get_fields(pic_sim* sim, void* const E[3], void* const B[3], void* const J[3], pic_mem where) {
  SIM_OR_FAIL(sim);
  return sim->impl->get_fields(E, B, J, where);
}

int pic_get_particles(pic_sim* sim, int32_t species, int64_t capacity, void* x, void* y, void* z, void* ux,
                      void* uy, void* uz, void* w, int64_t* id, int64_t* n_out, pic_mem where) {
  SIM_OR_FAIL(sim);
  void* out[7] = {x, y, z, ux, uy, uz, w};
  return sim->impl->get_particles(species, capacity, out, id, n_out, where);
}

int pic_get_sort_state(pic_sim* sim, int32_t species, int32_t* cell, int32_t* perm, pic_mem where) {
  SIM_OR_FAIL(sim);
  return sim->impl->get_sort_state(species, cell, perm, where);
}

int pic_sort_now(pic_sim* sim) {
  SIM_OR_FAIL(sim);
  return sim->impl->sort_now();
}

int pic_get_diagnostics(pic_sim* sim, double* out) {
  SIM_OR_FAIL(sim);
  return sim->impl->diagnostics(out);
}

int pic_get_rho(pic_sim* sim, double* rho, pic_mem where) {
  SIM_OR_FAIL(sim);
  return sim->impl->get_rho(rho, where);
}

int pic_enable_phase_timing(pic_sim* sim, int32_t on) {
  SIM_OR_FAIL(sim);
  return sim->impl->enable_timing(on);
}

int pic_get_phase_times(pic_sim* sim, float* ms, int64_t* spans, int32_t reset) {
  SIM_OR_FAIL(sim);
  return sim->impl->phase_times(ms, spans, reset);
}

int64_t pic_num_particles(const pic_sim* sim, int32_t species) {
  if (!sim || !sim->impl) return -1;
  return sim->impl->num_particles(species);
}

int32_t pic_num_species(const pic_sim* sim) {
  if (!sim || !sim->impl) return -1;
  return sim->impl->num_species();
}

const char* pic_last_error(const pic_sim* sim) {
  if (!sim || !sim->impl) return pic::g_create_error.c_str();
  return sim->impl->err.c_str();
}

int pic_ckc_coefficients(const double dx[3], double alpha[3], double beta[9], double gamma[3]) {
  if (!dx || !alpha || !beta || !gamma) return PIC_ERR_INVALID_ARG;
  for (int d = 0; d < 3; ++d)
    if (!(dx[d] > 0) || !std::isfinite(dx[d])) return PIC_ERR_INVALID_ARG;
  double be[3][3];
  pic::ckc_weights(dx, alpha, be, gamma);
  for (int a = 0; a < 3; ++a)
    for (int b = 0; b < 3; ++b) beta[3 * a + b] = be[a][b];
  return PIC_OK;
}

void pic_destroy(pic_sim* sim) {
  if (!sim) return;
  DeviceGuard device_guard_(sim->impl ? sim->impl->device : 0);
  delete sim->impl;
  delete sim;
}

}  // extern "C"
