// Host-side declarations shared by the translation units of libpic.so (CUDA path only).
#pragma once
#include <nvtx3/nvToolsExt.h>   // header-only NVTX v3
#include <cuda.h>   // CUtensorMap (types only: the encoder is fetched with cudaGetDriverEntryPoint, nothing links libcuda)

#include <set>
#include <string>
#include <vector>

#include "common.cuh"

namespace pic {

// Per-kernel-class device timers (pic_get_phase_times): CUDA events recorded on the simulation's
// stream around each launch group. Off unless enabled; recording never synchronises.
constexpr int kNumPhases = 5;   // == PIC_NPHASE: sort, push, deposit, stray, fields
struct Timer {
  struct Span { int phase; cudaEvent_t a, b; };
  bool on = false;
  std::vector<Span> spans;
  std::vector<cudaEvent_t> free_events;
  float ms[kNumPhases] = {0, 0, 0, 0, 0};
  int64_t count[kNumPhases] = {0, 0, 0, 0, 0};
  cudaEvent_t get_event() {
    if (!free_events.empty()) {
      cudaEvent_t e = free_events.back();
      free_events.pop_back();
      return e;
    }
    cudaEvent_t e;
    cudaEventCreate(&e);
    return e;
  }
  int begin(int phase, cudaStream_t st) {
    if (!on) return -1;
    Span sp{phase, get_event(), get_event()};
    cudaEventRecord(sp.a, st);
    spans.push_back(sp);
    return (int)spans.size() - 1;
  }
  void end(int idx, cudaStream_t st) {
    if (idx >= 0) cudaEventRecord(spans[idx].b, st);
  }
  void fold() {   // synchronises on the recorded events
    for (auto& s : spans) {
      cudaEventSynchronize(s.b);
      float t = 0;
      cudaEventElapsedTime(&t, s.a, s.b);
      ms[s.phase] += t;
      count[s.phase] += 1;
      free_events.push_back(s.a);
      free_events.push_back(s.b);
    }
    spans.clear();
  }
  void fold_completed() {   // folds the leading spans whose end event has already completed; never waits
    size_t k = 0;
    for (; k < spans.size(); ++k) {
      auto& s = spans[k];
      if (cudaEventQuery(s.b) != cudaSuccess) break;
      float t = 0;
      cudaEventElapsedTime(&t, s.a, s.b);
      ms[s.phase] += t;
      count[s.phase] += 1;
      free_events.push_back(s.a);
      free_events.push_back(s.b);
    }
    cudaGetLastError();   // cudaErrorNotReady is not an error here
    spans.erase(spans.begin(), spans.begin() + k);
  }
  void reset() {
    for (int i = 0; i < kNumPhases; ++i) { ms[i] = 0; count[i] = 0; }
  }
  void destroy() {
    for (auto& s : spans) { cudaEventDestroy(s.a); cudaEventDestroy(s.b); }
    for (auto e : free_events) cudaEventDestroy(e);
    spans.clear();
    free_events.clear();
  }
};

struct Ctx {
  cudaStream_t stream = nullptr;
  int device = 0;         // the device the handle was created on
  int sm_count = 148;     // its multiProcessorCount (grid sizing of the grid-stride kernels)
  std::set<const void*> smem_opted;   // kernels whose >48 KB dynamic shared memory opt-in is done for this handle
  // TMA staging of k_push_tile's E/B box (tile_kernels.cu make_push_tensor_map): one 4-D tensor map over the
  // six padded field arrays (x, y, z, component); off when the arrays do not meet TMA's 16-byte stride rule
  bool auto_deposit = true;   // pic_options.deposit_mode == AUTO: the library may pick a specialised kernel of the mode
  bool tma_push = false;
  alignas(64) CUtensorMap tmap_push;
  int64_t launches = 0;   // kernels launched through this handle
  Timer timer;
};

// times everything launched on c.stream during its lifetime as one span of `phase`, and brackets it with an
// NVTX range of the phase's name (the host-side launch window of each kernel class shows up
// in a timeline tool; NVTX v3 is header-only and does nothing when no tool is attached)
enum { kPhaseSort = 0, kPhasePush = 1, kPhaseDeposit = 2, kPhaseStray = 3, kPhaseFields = 4 };
inline const char* phase_name(int phase) {
  static const char* const names[kNumPhases] = {"pic:sort", "pic:gather+push", "pic:deposit", "pic:deposit(per-particle)",
                                                "pic:fields"};
  return phase >= 0 && phase < kNumPhases ? names[phase] : "pic";
}
struct ScopedPhase {
  Ctx& c;
  int idx;
  ScopedPhase(Ctx& c_, int phase) : c(c_), idx(c_.timer.begin(phase, c_.stream)) { nvtxRangePushA(phase_name(phase)); }
  ~ScopedPhase() {
    c.timer.end(idx, c.stream);
    nvtxRangePop();
  }
};

// ---- pic_api.cu: the text pic_last_error(NULL) returns, for handle-less entry points in other files
void set_handleless_error(const std::string& msg);

// ---- fields.cu
template <class R> void launch_push_B(const Grid<R>& g, const int lo[3], const int hi[3], Ctx& c);
template <class R> void launch_push_E(const Grid<R>& g, const int lo[3], const int hi[3], Ctx& c);
template <class R> void launch_fold_J(const Grid<R>& g, Ctx& c);
template <class R> void launch_fix_to_J(const Grid<R>& g, Ctx& c);   // deterministic deposition: fixed point -> J
template <class R> void launch_fill_guards(const Grid<R>& g, R* const* arrays, int narr, Ctx& c);
template <class R> void launch_pack(const Grid<R>& g, const R* valid_src, R* padded_dst, Ctx& c);
template <class R> void launch_unpack(const Grid<R>& g, const R* padded_src, R* valid_dst, Ctx& c);

// ---- particles.cu
enum { kDepositGlobal = 1, kDepositCoop = 2, kDepositTile = 3, kDepositTileMma = 4, kDepositFused = 5 };
// k_push_tile: threads per CTA (one CTA per tile). fp64: 12 warps per SM (two CTAs) already saturate the shared-memory
// path and 192 threads measured best (C2 push: 128: 1.672 ms, 160: 1.668, 192: 1.612, 224: 1.696, 256: 1.634, 320: 1.875);
// fp32 is latency-bound and wants the warps (C3: 0.316 ms at 256 against 0.331 at 192)
template <class R> constexpr int kPushTileThreads = sizeof(R) == 8 ? 192 : 256;
constexpr int kDepMmaWarps = 4;         // k_deposit_mma: warps per CTA (one CTA per tile) ...
constexpr int kDepMmaCtas = 5;          // ... and CTAs per SM the register budget is set for (20 warps per SM)
constexpr int kFusedWarps = 12;         // k_fused_mma: warps per CTA (one CTA per tile, one per SM: box + 12 record buffers = 216 KB)
constexpr int kFusedMaxDrift = 64;      // ... and the drifted particles each WARP lists for its second pass (12 x 64 x 4 B = 3 KB static)
constexpr int kDepTileWarps = 8;        // k_deposit_tile: warps per CTA (one CTA per tile, two per SM)
template <class R>
struct ParticleStep {
  Particles<R> cur;                  // x^n, u^{n-1/2}, w
  Particles<R> alt;                  // the other buffer set: its x,y,z receive x^{n+1} (COOP, TILE)
  const int32_t* cell_sorted;        // cell of every slot at the last sort, or nullptr
  const int32_t* tile_start;         // TILE: first slot of every tile (n_tiles + 1 entries)
  TileSpec tiles;
  int32_t* stray_list;               // scratch: indices a kernel hands to the next one (capacity n)
  unsigned int* stray_count;         // entries of stray_list
  unsigned long long* deactivated;
};
// One particle step of a species. Returns true if the new positions are in alt.{x,y,z}
// (the caller swaps the position pointers of the two buffer sets), false if updated in place.
template <class R>
bool launch_particles(const Grid<R>& g, const ParticleStep<R>& a, int order, int mode, Ctx& c);

// ---- tile_kernels.cu: the tensor map k_push_tile stages its box through (c.tma_push, c.tmap_push); false if
// TMA cannot describe these arrays (then the kernel copies element by element with cp.async). `stage_mode`:
// PIC_STAGE_* of pic_options (AUTO = TMA where it applies); tile_x = cells per tile along x.
template <class R>
bool make_push_tensor_map(const Grid<R>& g, int order, int tile_x, int stage_mode, Ctx& c);

// ---- tile_kernels.cu: the tile kernels of one species (needs tile_start): k_push_tile + k_deposit_tile /
// k_deposit_mma, or k_fused_mma (mode = kDepositTile / kDepositTileMma / kDepositFused); particles they
// could not finish are in stray_list / stray_count[0]
template <class R>
void launch_tile_kernels(const Grid<R>& g, const ParticleStep<R>& a, int order, int mode, Ctx& c);

// ---- sort.cu
struct SortScratch {
  uint32_t* keys[2] = {nullptr, nullptr};
  uint32_t* vals[2] = {nullptr, nullptr};
  uint32_t* hist = nullptr;       // 256 * nblocks digit histogram
  uint32_t* scan_tmp = nullptr;   // block sums of the scan (two levels)
  int64_t cap = 0;                // particles the buffers are sized for
  int64_t hist_len = 0;
  int64_t scan_len = 0;
  int32_t* stray_list = nullptr;  // particles.cu: indices handed from one deposition kernel to the next
  unsigned int* stray_count = nullptr;
};
int64_t sort_chunk();                                  // keys per block of a radix pass
int64_t sort_hist_len(int64_t n);                      // entries of `hist` for n particles
int64_t sort_scan_tmp_len(int64_t hist_len);           // entries of `scan_tmp`
// Stable sort of `cur` by tile-major cell key into `alt`; fills cell[], perm[] and (if not null)
// tile_start[n_tiles + 1], the first slot of every tile in the new order.
template <class R>
void sort_species(const Grid<R>& g, const TileSpec& t, const Particles<R>& cur, const Particles<R>& alt,
                  int32_t* cell, int32_t* perm, int32_t* tile_start, SortScratch& s, Ctx& c);

// ---- diag.cu
template <class R>
void launch_validate_particles(const Grid<R>& g, const Particles<R>& p, int* flags, Ctx& c);
template <class R>
void launch_validate_array(const R* a, int64_t n, int* flags, Ctx& c);
template <class R>
void launch_field_energy(const Grid<R>& g, double* out2, Ctx& c);              // out2[0]=sum E^2, [1]=sum B^2
template <class R>
void launch_particle_sums(const Particles<R>& p, double q, double m, double* out2, Ctx& c);  // KE, charge
template <class R>
void launch_max_abs(const R* a, int64_t n, double* out1, Ctx& c);   // *out1 = max(*out1, max |a|), out1 >= 0
template <class R>
void launch_rho(const Grid<R>& g, const Particles<R>& p, int order, double q, double* rho, Ctx& c);
template <class R>
void launch_gauss(const Grid<R>& g, const double* rho, double* out2, Ctx& c);  // max|divE-rho/eps0|, max|rho/eps0|

}  // namespace pic
