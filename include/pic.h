/* pic.h — C ABI of the B200-native electromagnetic PIC step (libpic.so).
 *
 * One call sequence runs the per-step particle loop of the electromagnetic PIC method that
 * arXiv 2101.12149 ("Porting WarpX to GPU-accelerated platforms") ports to GPUs:
 *   cell-tile particle sort      (§3.4.2 "Particle Sorting")
 *   fused field gather + push    (§3.1: fields re-gathered inside the push kernel)
 *   Esirkepov current deposition (§3.4.1; ref [8] PAPER.md:301)
 *   Yee FDTD update of E and B   (§2.4: B on faces, E and J on edges; ref [28])
 *   guard-cell sum and fill      (§2.4 FillBoundary / SumBoundary)
 * on ONE GPU, one periodic (or z-truncated) box. The formulas are fixed in DESIGN.md
 * ("The step", "Readings"); every step runs in hand-written CUDA kernels for sm_100a.
 * There is no CPU fallback: every call fails with PIC_ERR_CUDA when no device is usable.
 *
 * Conventions
 *  - Units: SI. Positions in metres inside [0, n_cells[d]*dx[d]); momenta u = gamma*v in m/s;
 *    weight = real particles per macro-particle; E in V/m, B in T, J in A/m^2.
 *  - Element type of every `void*` array is double under PIC_F64 and float under PIC_F32.
 *  - Fields: one array per component holding n_x*n_y*n_z values of the valid region, x fastest
 *    (idx = i + n_x*(j + n_y*k), "Fortran index order"); guard cells are internal.
 *    Array element [i,j,k] of a component is the value at its Yee location:
 *      Ex,Jx (i+1/2,j,k)  Ey,Jy (i,j+1/2,k)  Ez,Jz (i,j,k+1/2)
 *      Bx (i,j+1/2,k+1/2) By (i+1/2,j,k+1/2) Bz (i+1/2,j+1/2,k)
 *  - Particles: structure of arrays, one array per attribute.
 *  - `where` says whether the caller's pointers are host (PIC_HOST) or device (PIC_DEVICE)
 *    memory. The library copies every input during the call (the caller may free at once) and
 *    writes outputs into caller-allocated buffers. Scalars and small structs are host memory.
 *  - Time levels: supplied u is u^{n-1/2}; supplied x, E, B are at time n. No back-push.
 *  - Every call returns 0 or a negative PIC_ERR_*; nothing throws or aborts across the ABI.
 *    pic_step is asynchronous on the simulation's stream; asynchronous faults surface at the
 *    next synchronising call (pic_get_*, pic_synchronize).
 *  - A pic_sim is not thread-safe; use one host thread per handle.
 */
#ifndef PIC_H_
#define PIC_H_

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#if defined(__GNUC__)
#define PIC_API __attribute__((visibility("default")))
#else
#define PIC_API
#endif

typedef struct pic_sim pic_sim; /* opaque; created by pic_create, freed by pic_destroy */

typedef enum { PIC_F64 = 0, PIC_F32 = 1 } pic_precision;
typedef enum { PIC_HOST = 0, PIC_DEVICE = 1 } pic_mem;

enum {
  PIC_OK = 0,
  PIC_ERR_INVALID_ARG = -1,   /* null pointer, order not in 1..3, tile does not divide, n < 0, NaN/Inf input */
  PIC_ERR_CFL = -2,           /* dt*c*sqrt(sum 1/dx^2) > 1 */
  PIC_ERR_OUT_OF_DOMAIN = -3, /* a particle position outside [0, L) */
  PIC_ERR_OOM = -4,           /* device allocation failed */
  PIC_ERR_CUDA = -5,          /* CUDA error (text in pic_last_error), or no CUDA device */
  PIC_ERR_CAPACITY = -6       /* caller's output buffer too small */
};

/* Deposition kernels: all compute the same sums in a different order. */
enum {
  PIC_DEPOSIT_AUTO = 0,       /* library's choice for the precision / order / sort state */
  PIC_DEPOSIT_GLOBAL = 1,     /* one thread per particle, one global atomic per particle-node
                                 (the paper's GPU design) */
  PIC_DEPOSIT_COOP = 2,       /* warp-cooperative: a warp walks its particles, lanes own window
                                 nodes, sums held in registers per cell run, one global
                                 reduction per node and run */
  PIC_DEPOSIT_TILE = 3,       /* one CTA per sort tile (tile edges <= 8 cells, after the first
                                 sort; otherwise falls back to COOP / GLOBAL): E/B stencil box
                                 staged in shared memory for gather + push; deposition by
                                 16-lane groups (4 at order 1) that own the (j,k) columns of a
                                 cell's window, sums in registers, one L2 reduction per finished
                                 window node. AUTO picks this in fp32 when it can; at order 1 AUTO
                                 (not an explicit TILE) deposits through the tile's J box in shared
                                 memory instead: lane = particle, segmented warp reduction per cell
                                 run, native fp32 shared-memory reductions, one flush per tile. */
  PIC_DEPOSIT_TILE_MMA = 4,   /* as TILE, but the sums of a cell's particles are formed as small
                                 dense contractions on the fp64 tensor pipe (mma.sync m8n8k4.f64),
                                 one warp per cell run (fp64 arithmetic also for PIC_F32 data).
                                 AUTO picks this in fp64 when it can. */
  PIC_DEPOSIT_FUSED = 5       /* gather + push + the TILE_MMA deposition in ONE kernel per species: a
                                 warp takes 32 particles through the whole particle step, so x_old,
                                 x_new, w and the nodal weights reach the deposit in registers and
                                 shared memory instead of through HBM. fp64 only (PIC_F32 runs TILE).
                                 Measured slower than TILE_MMA's two kernels on B200 (one CTA of 12
                                 warps per SM against 16 + 20 warps): kept
                                 selectable, never picked by AUTO. */
};

/* Momentum update of step 2c. BORIS: the relativistic Boris rotation (BASELINE.json; DESIGN.md
 * reading Q2). VAY: the Vay pusher the paper's LWFA run uses (ref [21]; SURVEY.md
 * 8(f) NEXT-4): u' = u + 2 kq E + kq (u/gamma) x B, then the closed-form gamma and rotation. */
enum { PIC_PUSHER_BORIS = 0, PIC_PUSHER_VAY = 1 };

/* Field gather of step 2b. UNIFORM: order n on every axis, each component from its own staggered
 * location (reading Q1). GALERKIN: order n-1 along every axis on which the component is
 * staggered ("energy-conserving" gather). */
enum { PIC_GATHER_UNIFORM = 0, PIC_GATHER_GALERKIN = 1 };

/* Field solver of steps 3-5. YEE: the standard Yee curl (ref [28]); time step limit
 * dt*c*sqrt(sum 1/dx^2) <= 1. CKC: Cole-Karkkainen-Cowan (ref [12]): the E
 * update is Yee's, every difference of E in the B update is smoothed over the 3x3 transverse
 * neighbours with the weights alpha, beta, gamma of DESIGN.md section 11; no dispersion along the
 * axes at c*dt = min(dx), which is also its time step limit (PIC_ERR_CFL beyond it). */
enum { PIC_SOLVER_YEE = 0, PIC_SOLVER_CKC = 1 };

/* How k_push_tile brings a tile's E/B stencil box into shared memory (north_star: "TMA where the box is
 * regular"; PAPER.md:209-211 contrasts the paper's cached global reads with explicit shared-memory staging).
 * AUTO: one bulk tensor copy per CTA (cp.async.bulk.tensor, TMA) in fp64 whenever the padded field arrays
 * meet TMA's 16-byte stride rule (even padded extents), else element-wise cp.async. CP_ASYNC / TMA force one
 * (TMA silently falls back where the rule is not met). Results are bit-identical either way. */
enum { PIC_STAGE_AUTO = 0, PIC_STAGE_CP_ASYNC = 1, PIC_STAGE_TMA = 2 };

/* Options; pass NULL to pic_create for the defaults given here. */
typedef struct {
  int32_t periodic[3];   /* default {1,1,1}; 0 = truncation with zeroed guard cells on that axis:
                            fields outside read 0, J deposited outside is dropped, a particle
                            leaving through it is deactivated (weight := 0) */
  int32_t tile[3];       /* cells per sort tile, default {8,8,8}; each must divide n_cells (a tile
                            larger than the grid is clipped to the grid) */
  int32_t sort_interval; /* sort every this many steps, first at step 0; default 4
                            (PAPER.md:201); 0 = never */
  int32_t sort_key_mode; /* 0 = tile-major cell key (default): tile index major, cell inside
                            the tile minor; 1 = tile index only */
  int32_t deposit_mode;  /* PIC_DEPOSIT_*; default PIC_DEPOSIT_AUTO */
  int32_t pusher;        /* PIC_PUSHER_*; default PIC_PUSHER_BORIS */
  int32_t gather_mode;   /* PIC_GATHER_*; default PIC_GATHER_UNIFORM */
  int32_t solver;        /* PIC_SOLVER_*; default PIC_SOLVER_YEE */
  int32_t deterministic; /* 0 (default): J is summed with floating-point reductions at L2, in whatever
                            order the warps arrive, so J differs from run to run in
                            the last bits. 1: every contribution is split into two 64-bit fixed-point
                            parts and summed with INTEGER reductions, which are associative: J, and with
                            it the whole simulation, is bit-identical from run to run (SURVEY.md 8(f)
                            NEXT-1, "atomic-order-free deposition"). Any deposit_mode. Costs a second
                            reduction per contribution and 48 bytes per grid node. */
  int32_t cuda_graph;    /* 1 (default): pic_step captures each time step once per buffer arrangement
                            (they repeat with period 2 x sort_interval) and replays it as ONE graph launch
                            (launch latency dominates once the kernels are fast). The first
                            step of a handle, and every step while phase timing is on, is launched kernel
                            by kernel. 0: always kernel by kernel. Results are identical either way. */
  int32_t box_staging;   /* PIC_STAGE_*; default PIC_STAGE_AUTO */
  void*   cuda_stream;   /* cudaStream_t all work is issued on (e.g. torch's current stream);
                            NULL = the legacy default stream */
} pic_options;

/* Fill *opt with the defaults. */
PIC_API void pic_default_options(pic_options* opt);

/* A handle belongs to the CUDA device that is current when pic_create is called; every later call on it
 * makes that device current for its duration and restores the caller's device before returning.
 *
 * Create a simulation on the current CUDA device: a box of n_cells[3] Yee cells of size dx[3]
 * (metres), time step dt (seconds), B-spline shape order 1..3 used for both gather and deposit,
 * working precision prec. Fields start at zero. *out receives the handle.
 * Limits: field nodes are indexed with 32 bits, (n_cells + 8)^3 padded nodes must stay below 2^31
 * (INVALID_ARG otherwise), and the sort key (tiles x cells per tile) below 2^32.
 * Errors: INVALID_ARG, CFL, OOM, CUDA. */
PIC_API int pic_create(const int32_t n_cells[3], const double dx[3], double dt, int shape_order,
               pic_precision prec, const pic_options* opt, pic_sim** out);

/* Add a species of n macro-particles (one container per species) with charge (C)
 * and mass (kg) per real particle. x..w are arrays of n elements in `where` memory. Particle ids
 * are 0..n-1 in the order given and follow the particles through every sort. *species_id
 * (nullable) receives the species index (0,1,...). Species are processed in insertion order.
 * Limit: particle slots are indexed with 32 bits inside the kernels (tile_start[], the stray list,
 * perm[]), so n < 2^31 per species (INVALID_ARG otherwise); the number of species is not limited.
 * Errors: INVALID_ARG (incl. non-finite values), OUT_OF_DOMAIN, OOM, CUDA. Synchronises. */
PIC_API int pic_add_species(pic_sim* sim, int64_t n, const void* x, const void* y, const void* z,
                    const void* ux, const void* uy, const void* uz, const void* w,
                    double charge, double mass, pic_mem where, int32_t* species_id);

/* Overwrite E and B (valid region, layout above) and refresh the guard cells. E, B: arrays of
 * three pointers. Errors: INVALID_ARG (incl. non-finite), CUDA. Synchronises. */
PIC_API int pic_set_fields(pic_sim* sim, const void* const E[3], const void* const B[3], pic_mem where);

/* Advance n steps: per step, per species { sort if due } -> zero J -> per species
 * { gather + Boris push + Esirkepov deposit + wrap } -> sum J guards -> B half step -> E full
 * step -> B half step -> fill E/B guards. Asynchronous. */
PIC_API int pic_step(pic_sim* sim, int32_t n);

/* Block until all issued work is done; returns PIC_ERR_CUDA if any of it faulted. */
PIC_API int pic_synchronize(pic_sim* sim);

/* Copy the valid region of E, B and (if J != NULL) the J of the last step into the caller's
 * arrays (three pointers each, n_x*n_y*n_z elements). Any of E, B, J may be NULL. Synchronises. */
PIC_API int pic_get_fields(pic_sim* sim, void* const E[3], void* const B[3], void* const J[3], pic_mem where);

/* Copy species `species` in its CURRENT internal order into caller arrays of `capacity`
 * elements (any pointer may be NULL to skip that attribute); *n_out (nullable) = particle count.
 * Errors: INVALID_ARG, CAPACITY. Synchronises. */
PIC_API int pic_get_particles(pic_sim* sim, int32_t species, int64_t capacity, void* x, void* y, void* z,
                      void* ux, void* uy, void* uz, void* w, int64_t* id, int64_t* n_out, pic_mem where);

/* State of the most recent sort of a species: cell[k] = linear cell index
 * (c_x + n_x*(c_y + n_y*c_z)) of the particle in slot k right after that sort, perm[k] = slot
 * the particle held before it. Either pointer may be NULL. Errors: INVALID_ARG (never sorted). */
PIC_API int pic_get_sort_state(pic_sim* sim, int32_t species, int32_t* cell, int32_t* perm, pic_mem where);

/* Sort every species now (the same operation pic_step runs when a sort is due). Asynchronous. */
PIC_API int pic_sort_now(pic_sim* sim);

/* Diagnostics, reduced on the device in fp64 (host array of PIC_NDIAG doubles). Synchronises. */
enum {
  PIC_DIAG_FIELD_E = 0,     /* 1/2 eps0 sum E^2 dV  [J] */
  PIC_DIAG_FIELD_B = 1,     /* 1/2 eps0 c^2 sum B^2 dV [J] */
  PIC_DIAG_KINETIC = 2,     /* sum w m c^2 (gamma-1) over all species, at the stored u [J] */
  PIC_DIAG_CHARGE = 3,      /* sum q w [C] */
  PIC_DIAG_GAUSS_MAX = 4,   /* max |div E - rho/eps0|, rho from the order-n nodal shape */
  PIC_DIAG_RHO_MAX = 5,     /* max |rho/eps0| */
  PIC_DIAG_DEACTIVATED = 6, /* particles deactivated at a non-periodic boundary so far */
  PIC_DIAG_STEPS = 7,       /* steps taken */
  PIC_DIAG_POOL_CHUNKS = 8, /* cudaMalloc calls made by the memory pool so far */
  PIC_DIAG_POOL_BYTES = 9,  /* bytes held by the pool */
  PIC_DIAG_LAUNCHES = 10,   /* kernels launched by this handle so far (all calls) */
  PIC_DIAG_STEP_LAUNCHES = 11, /* kernels launched by pic_step and pic_sort_now so far */
  PIC_NDIAG = 12
};
PIC_API int pic_get_diagnostics(pic_sim* sim, double* out);

/* Nodal charge density rho (C/m^3, fp64, n_x*n_y*n_z, x fastest) of all species. Synchronises. */
PIC_API int pic_get_rho(pic_sim* sim, double* rho, pic_mem where);

/* Device time per kernel class, from CUDA events recorded on the simulation's stream around each
 * launch group (never synchronises while stepping). ms[p] = elapsed time (ms) summed over the
 * spans of class p since the last call with reset != 0, spans[p] (nullable) = how many spans that
 * was (one span = one launch of that class's kernel for PUSH / DEPOSIT / STRAY, one whole sort
 * for SORT, one launch group for FIELDS). Host arrays of PIC_NPHASE elements. Timing is off
 * until pic_enable_phase_timing(sim, 1). pic_get_phase_times synchronises. */
enum {
  PIC_PHASE_SORT = 0,    /* keys, radix passes, permutation of all attributes */
  PIC_PHASE_PUSH = 1,    /* gather + momentum push (+ deposit when PIC_DEPOSIT_GLOBAL fuses it) */
  PIC_PHASE_DEPOSIT = 2, /* Esirkepov deposition of the sorted runs (tensor-pipe / lane-group / warp-cooperative kernel) */
  PIC_PHASE_STRAY = 3,   /* per-particle deposition of the particles that kernel listed instead */
  PIC_PHASE_FIELDS = 4,  /* J zero, J guard sum, Yee B/E/B, guard fill */
  PIC_NPHASE = 5
};
PIC_API int pic_enable_phase_timing(pic_sim* sim, int32_t on);
PIC_API int pic_get_phase_times(pic_sim* sim, float* ms, int64_t* spans, int32_t reset);

PIC_API int64_t pic_num_particles(const pic_sim* sim, int32_t species); /* < 0 on error */
PIC_API int32_t pic_num_species(const pic_sim* sim);

/* Text of the last error of this handle ("" if none). sim == NULL: the last pic_create error.
 * The string is owned by the library and valid until the next call on the same handle. */
PIC_API const char* pic_last_error(const pic_sim* sim);

/* On-chip ceilings of the current CUDA device, measured now: the roofline method of the paper quotes
 * kernels against MEASURED ceilings (Fig. 2), and the two units that bound the
 * particle kernels here (the fp64 pipe and shared-memory bandwidth) are in no vendor or driver file.
 * Each probe (a register-resident loop filling every warp slot of every SM) is launched on `cuda_stream`
 * (NULL = legacy default) repeatedly for at least `seconds_per_probe` seconds (and at least 3 times); the
 * best launch is reported. out: host array of PIC_NPROBE doubles. No simulation handle is involved and no
 * PIC work is done. Synchronises. Errors: INVALID_ARG, CUDA. */
enum {
  PIC_PROBE_FP64_FMA_TFLOPS = 0, /* DFMA, 8 independent chains per thread */
  PIC_PROBE_FP64_MMA_TFLOPS = 1, /* mma.sync.m8n8k4.f64 (the deposit's tensor-pipe instruction), 2 flop per FMA */
  PIC_PROBE_SMEM_TBS = 2,        /* conflict-free 64-bit shared-memory loads, TB/s */
  PIC_PROBE_FP32_FMA_TFLOPS = 3, /* FFMA, 16 independent chains per thread */
  PIC_PROBE_SM_COUNT = 4,        /* multiprocessors of the device */
  PIC_PROBE_SM_CLOCK_MHZ = 5,    /* the device's nominal maximum SM clock (cudaDevAttrClockRate) */
  PIC_NPROBE = 6
};
PIC_API int pic_probe_peaks(void* cuda_stream, double seconds_per_probe, double* out);

/* The weights the CKC solver (PIC_SOLVER_CKC, ref [12]) uses for cells of size dx[3]: the difference of
 * E along axis a in the B update is alpha[a]*dF(0,0) + beta[3a+b]*[dF(+b) + dF(-b)] + beta[3a+c]*[dF(+c) +
 * dF(-c)] + gamma[a]*[the four corners] over the 3x3 transverse neighbours (b, c the other two axes;
 * beta[3a+a] = 0). Host arithmetic only, no device needed (lets the weights be checked against what they
 * are built for: unit sum, stability at c*dt = min(dx), no dispersion along the axes). Host pointers:
 * alpha[3], beta[9], gamma[3]. Errors: INVALID_ARG. */
PIC_API int pic_ckc_coefficients(const double dx[3], double alpha[3], double beta[9], double gamma[3]);

/* The sort of step 1 for callers that may NOT allocate: code under
 * CUDA graph capture, tight serving loops, harnesses that forbid cudaMalloc. Computes, for n particles at
 * positions x, y, z, exactly what pic_sort_now + pic_get_sort_state give — perm[k] = the input slot of the
 * particle that the stable sort by tile-major cell key puts at slot k, cell[k] = its cell index
 * cx + Nx*(cy + Ny*cz) — with the same kernels, and makes no cudaMalloc / cudaFree / pool call: the scratch of
 * the radix passes is ONE file-scope device array of fixed size inside the library (about 8.3 MB, held by every
 * GPU that loads the library until the process exits). Hence the limit n <= PIC_NOALLOC_MAX_PARTICLES
 * (PIC_ERR_CAPACITY beyond it, with a message in pic_last_error(NULL)).
 * x, y, z, cell, perm are DEVICE pointers (elements of prec; int32 outputs of n entries); n_cells, dx, tile are
 * host arrays with the meaning they have in pic_create / pic_options (a tile larger than the grid is clipped).
 * No particle data is moved; no handle is involved. Asynchronous on cuda_stream (NULL = the legacy default
 * stream); runs on the current device. All calls on one device share the scratch array: two calls that overlap
 * on the GPU (different streams without a dependency) race — order them. Nothing is kept between calls.
 * Errors: INVALID_ARG, CAPACITY, CUDA. */
#define PIC_NOALLOC_MAX_PARTICLES 524288
PIC_API int pic_sort_permutation_noalloc(const int32_t n_cells[3], const double dx[3], const int32_t tile[3],
                                         int32_t sort_key_mode, pic_precision prec, const void* x, const void* y,
                                         const void* z, int64_t n, int32_t* cell, int32_t* perm, void* cuda_stream);

/* Free everything the handle owns (synchronises). NULL is a no-op. */
PIC_API void pic_destroy(pic_sim* sim);

#ifdef __cplusplus
}
#endif
#endif /* PIC_H_ */
