/*
 * ljmd.h -- C ABI of the B200-native Lennard-Jones MD hot path of arXiv 0709.3225
 * ("Harvesting graphics power for MD simulations"): one velocity-Verlet step with the
 * force evaluated as all-pairs O(N^2) or through a cell list, and the rand48 generator
 * with skip-ahead.  Citations are PAPER.md:<line> in /root/reference; "R<n>" are the
 * numbered readings in DESIGN.md section 3.
 *
 * Conventions for every call
 *   - Returns MD_OK (0) or a negative md_status; never aborts, never throws.
 *   - Every array pointer is owned by the caller, may be HOST or DEVICE memory (detected
 *     with cudaPointerGetAttributes), and is not retained after the call returns.
 *   - Calls are synchronous for the caller: results are complete on return.  Kernels run
 *     on the stream set with md_set_stream (default: the legacy default stream; the Python
 *     binding's md_create sets PyTorch's current stream and allocator instead, unless it is
 *     called with torch_plumbing=False).
 *   - A handle is not thread-safe; distinct handles are independent.
 *   - Everything executes on the current CUDA device in sm_100a kernels.  There is no CPU
 *     fallback: without a usable device every call returns MD_ECUDA.
 *   - Reduced units, mass = 1, cubic periodic box [0,L)^3, minimum image (R3).
 */
#ifndef LJMD_H
#define LJMD_H

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct md_sim md_sim; /* opaque, created and destroyed by the library */

typedef enum md_status {
    MD_OK = 0,
    MD_EINVAL = -1,       /* null pointer, non-positive size, unknown enum, rc > L/2, bad seed */
    MD_EDOMAIN = -2,      /* algo = MD_CELL with fewer than 3 cells per dimension */
    MD_ESTATE = -3,       /* step/get before md_set_state, or getters on stale forces */
    MD_ENOMEM = -4,       /* device or host allocation failed */
    MD_ECUDA = -5,        /* CUDA runtime error; see md_last_cuda_error */
    MD_EUNSUPPORTED = -6  /* valid request that this build does not implement */
} md_status;

/* algo.  MD_VERLET (an extension beyond the paper's two algorithms; it discusses neighbour lists in
 * PAPER.md:100-104): neighbour lists with a skin, built from a cell list of side >= rc + skin and rebuilt,
 * on the device's own decision, whenever an atom has moved more than skin / 2 since the last build.  Same
 * forces as the other two paths; MD_EDOMAIN if int[L / (rc + skin)] < 3, MD_EUNSUPPORTED if N > 2^23 - 1.
 * Lists start with room for 1.4 x the mean length + 32 entries and are never truncated silently: a build
 * that needs more makes md_compute_forces (and the evaluation md_step does on stale forces) reallocate them
 * for the length asked for and rebuild; if that happens in the middle of md_step, the call returns MD_ENOMEM,
 * the forces and the trajectory since that build are not valid (set the state again; the lists have been
 * enlarged for the next attempt). */
enum { MD_ALLPAIRS = 0, MD_CELL = 1, MD_VERLET = 2 };
enum { MD_TRUNCATED = 0, MD_ENERGY_SHIFTED = 1, MD_FORCE_SHIFTED = 2 }; /* shifted */
enum { MD_POT_LJ = 0, MD_POT_YUKAWA = 1 };                                /* md_set_potential */
enum { R48_U32_HI32 = 0, R48_U32_HI31 = 1, R48_F64 = 2, R48_U64_STATE = 3 }; /* kind */

/* Create a simulation of N atoms in a cubic periodic box of side L with the Lennard-Jones
 * pair force of PAPER.md:56 (Eq. 2, with the 1/sigma factor of R1) cut at rc (strict r < rc,
 * PAPER.md:61).  shifted: 0 truncated only; 1 energy-shifted, U(rc) = 0, force unshifted
 * (the graded mode, R2); 2 the paper's force-shifted Eq. 3.  dt is the
 * velocity-Verlet time step.  The box used is (double)(float)L (R13).
 * Errors: MD_EINVAL for out == NULL, N <= 0, L <= 0, rc <= 0, eps < 0, sigma <= 0, dt <= 0,
 * unknown shifted, or rc > L/2 (minimum image invalid); MD_ENOMEM; MD_ECUDA. */
int md_create(md_sim **out, int64_t N, double L, double rc, double eps, double sigma,
              double dt, int shifted);

/* Free the handle and all device memory it owns.  md_destroy(NULL) is MD_OK. */
int md_destroy(md_sim *s);

/* Set positions and velocities, [N][3] floats xyz, host or device.  Positions are wrapped
 * into [0,L) (R14).  Marks forces stale.  Atom i of these arrays is "atom i" for every
 * getter, whatever internal order the library keeps. */
int md_set_state(md_sim *s, const float *pos, const float *vel);

/* Read back positions and velocities in the caller's atom order; either may be NULL. */
int md_get_state(md_sim *s, float *pos, float *vel);

/* Evaluate F, PE and the virial at the current positions with the given algo, without
 * stepping (Eq. 1; PAPER.md:98-112 for MD_CELL).  Also refreshes KE.
 * MD_EDOMAIN if algo = MD_CELL and int[L/rc] < 3. */
int md_compute_forces(md_sim *s, int algo);

/* Advance nsteps velocity-Verlet steps (order per R4): half-kick, drift with
 * periodic wrap, force evaluation with algo, half-kick.  If the forces are stale they are
 * evaluated first with algo; that evaluation is not a step.  Forces last evaluated by another
 * algo are reused as they are (all paths compute the same forces) except by the paths whose
 * integrator needs their own data layout: MD_VERLET, and MD_CELL with "cell_skin", evaluate
 * first when another path ran last.  MD_CELL rebuilds the cell list from current positions
 * before every force evaluation (R20; "cell_skin" = 0).  nsteps = 0 is allowed.  Atoms moving more than L per step and
 * coincident atoms are undefined behaviour. */
int md_step(md_sim *s, int64_t nsteps, int algo);

/* Maxwell-Boltzmann start velocities on the device (an extension: SURVEY 8(f) item 3; the paper names
 * rand48 as the generator for such uses).  One rand48 stream started at state
 * seed48 (< 2^48); atom i (caller's order) consumes draws 6 i .. 6 i + 5: per component u1, u2 and
 * v = sqrt(T) sqrt(-2 ln(1 - u1)) cos(2 pi u2); then the mean is removed and the set rescaled so that
 * sum v^2 = 3 N T; stored as FP32.  Needs md_set_state first (MD_ESTATE); positions and forces are
 * untouched, KE is refreshed.  MD_EINVAL: T <= 0, seed48 >= 2^48, N < 2. */
int md_init_velocities(md_sim *s, double T, uint64_t seed48);

/* Forces [N][3] at the current positions, caller's atom order.  MD_ESTATE if stale. */
int md_get_forces(md_sim *s, float *f);

/* KE = (1/2) sum v^2, PE = sum_{i<j} U(r_ij), virial = sum_{i<j} r_ij f(r_ij) (R12), all at
 * the current time; any pointer may be NULL.  MD_ESTATE if forces are stale. */
int md_get_energies(md_sim *s, double *KE, double *PE, double *virial);

/* rand48 (Eq. 5): x <- (0x5DEECE66D x + 0xB) mod 2^48; each output is
 * taken from the NEW state (R8).  seeds[s] is the 48-bit state of stream s (bits 48..63 must
 * be zero) and is replaced by the state after ndraws draws, so consecutive calls concatenate
 * bit-exactly.  Output is stream-major: out[s*ndraws + d] is draw d of
 * stream s.  kind: 0 uint32 x>>16; 1 uint32 x>>17 (lrand48); 2 double x*2^-48; 3 uint64 x.
 * Streams are split across warps by O(log k) skip-ahead (Eq. 6-7 with
 * R5), so nstreams = 1 with a large ndraws runs on the whole GPU.  seeds and out may each be
 * host or device memory.  ndraws = 0 or nstreams = 0 is MD_OK and writes nothing.
 * MD_EINVAL for a seed with bits above 47 (host seeds are checked before anything runs; device seeds by the
 * generating kernel itself, so the answer comes at the end of the call): no seed is changed, the contents of
 * `out` are then unspecified. */
int rand48_fill(uint64_t *seeds, int64_t nstreams, int64_t ndraws, int kind, void *out);

/* Human-readable name of a status code; never NULL. */
const char *md_strerror(int code);

/* ---- helpers (not named by the paper; needed by tests, bench and bindings) ---- */

/* Stream (a cudaStream_t passed as void*) on which this handle's kernels run. */
int md_set_stream(md_sim *s, void *cuda_stream);
/* Another pair potential through the same machinery (an extension: PAPER.md:184, Outlook, "it is trivial to
 * replace this potential by other pair-potentials, including the coulombic interaction").
 *   MD_POT_LJ      Lennard-Jones with the eps, sigma of md_create (a, b ignored); the default.
 *   MD_POT_YUKAWA  screened Coulomb between equal charges, U(r) = a exp(-b r) / r, f = -dU/dr
 *                  (b = 0: the bare Coulomb pair a / r), truncated at the rc of md_create, with the same
 *                  meaning of `shifted` (1: U - U(rc); 2: f - f(rc) and the matching U).  Every in-range
 *                  pair is evaluated in FP64 on all three force paths (the FP32 fast branch of the cell and
 *                  neighbour-list kernels exists for Lennard-Jones only, so those paths run slower).
 * Marks the forces stale.  MD_EINVAL for an unknown kind, non-finite a or b, or b < 0. */
int md_set_potential(md_sim *s, int kind, double a, double b);

/* All-pairs forces, PE and virial WITHOUT any device allocation: for callers that cannot call cudaMalloc.
 * That is a process whose memory pool took the whole card at start-up (a cudaMalloc made by a library then
 * fails), or a loop with a latency budget, where cudaMalloc / cudaFree are ruled out because they stall the
 * whole device.  md_create and the calls on a handle do allocate; this one call never does.
 *
 * Computes what md_compute_forces(MD_ALLPAIRS) computes (Eq. 1, with the Lennard-Jones pair
 * of PAPER.md:56-61 and the same meaning of rc, eps, sigma, shifted as md_create; every in-range pair in
 * FP64; box (double)(float)L, minimum image): forces[i] = F_i, pe_virial[0] = sum_{i<j} U,
 * pe_virial[1] = sum_{i<j} r f.  Stateless: no handle, no velocities, Lennard-Jones only.
 *   pos        [N][3] floats, DEVICE memory, read only, expected in [0, L) (used as given, not wrapped)
 *   forces     [N][3] floats, DEVICE memory, overwritten, same atom order as pos
 *   pe_virial  2 doubles,     DEVICE memory, overwritten
 * All three stay the caller's; host pointers are refused (MD_EINVAL), since staging them would need an
 * allocation.  Runs on cuda_stream (a cudaStream_t; NULL = legacy default stream) and returns after that
 * stream has finished the work, like every other call here.
 *
 * Scratch: the partial sums of the kernel live in one array built into the library, about 1.3 MB, which each
 * GPU that loads the library keeps until the process exits.  Its fixed size sets the limit
 * N <= MD_STATIC_MAX_ATOMS; a larger N returns MD_EUNSUPPORTED and nothing is launched.  Every call on a
 * device shares that array (it keeps the previous call's contents; what must start at zero is cleared by each
 * call itself), so calls that overlap on the GPU -- two host threads, two streams -- race with each other:
 * serialise them.  The first call on each device looks up the array's device address
 * (cudaGetSymbolAddress, with that device current); make that first call before starting any stream capture.
 * Errors: MD_EINVAL as md_create, plus NULL or non-device pointers; MD_EUNSUPPORTED; MD_ECUDA. */
#define MD_STATIC_MAX_ATOMS 16384
int md_forces_allpairs_static(const float *pos, int64_t N, double L, double rc, double eps, double sigma,
                              int shifted, float *forces, double *pe_virial, void *cuda_stream);

/* The same on an explicit CUDA stream (no process-wide state involved). */
int rand48_fill_on(uint64_t *seeds, int64_t nstreams, int64_t ndraws, int kind, void *out, void *cuda_stream);

/* Stream used by rand48_fill (process-wide; rand48_fill_on takes the stream per call instead). */
int rand48_set_stream(void *cuda_stream);

/* Device allocator hooks (process-wide), e.g. PyTorch's caching allocator.  alloc returns a
 * device pointer or NULL; both are called with the stream in use.  NULL, NULL restores
 * cudaMalloc/cudaFree.  May be changed at any time: every block is released through the hook
 * that was installed when it was allocated. */
typedef void *(*md_alloc_fn)(int64_t bytes, void *cuda_stream);
typedef void (*md_free_fn)(void *ptr, void *cuda_stream);
int md_set_allocator(md_alloc_fn alloc, md_free_fn free_);

/* Tuning and introspection.  md_set_option keys:
 *   "graph"          1 (default): inside one md_step call the interior steps (all but the first and
 *                    the last) are replayed from a CUDA graph that holds one unit of steps (2 on the
 *                    cell path, 2 * sort_every on the sorted all-pairs path: the number of steps
 *                    after which the buffer roles repeat); 0 = launch every kernel directly
 *   "andersen_nu", "andersen_T", "andersen_seed"
 *                    Andersen thermostat (an extension: SURVEY 8(f) item 3; thermostats are among the uses
 *                    the paper names for its generator): after the second
 *                    half-kick of every step each atom takes, with probability nu * dt (as the 32-bit
 *                    threshold floor(nu dt 2^32), md_get_stat "andersen_threshold"), a fresh velocity
 *                    sqrt(T) sqrt(-2 ln(1 - u1)) cos(2 pi u2) per component.  One rand48 stream from state
 *                    "andersen_seed" (< 2^48); step t since the last change of these options and atom i
 *                    own draws 7 (t N + i) .. + 6 (the first decides, by integer comparison of its 32
 *                    high bits).  Active once nu > 0 and T > 0; nu = 0 switches it off.  Steps are then
 *                    launched directly (no graph, no folded half-kick).
 *   "skin"           MD_VERLET: list radius minus rc (default 0.3 sigma); only before the first use
 *   "cell_skin"      MD_CELL on skin cells: cells of side >= rc + value, re-sorted on the device's own
 *                    decision when an atom has strayed value / 2; 0 (default) = the cell
 *                    list is rebuilt every step.  Shares the skin with MD_VERLET (set before either runs)
 *   "vl_fuse"        1 (default): interior steps of md_step(MD_VERLET) integrate in the epilogue of the list
 *                    force kernel (full lists only); 0 = separate integration kernel
 *   "vl_half"        MD_VERLET with half lists: every pair once, the reaction force through vector
 *                    reductions (default 0; measured in DESIGN.md section 7b)
 *   "cell_group"     cells of one z-column handled by one warp of the cell-force kernel (1..5);
 *                    0 (default) = chosen from the mean occupancy
 *   "time_kernels"   1 = record CUDA events around every phase of md_step (disables the graph);
 *                    read back with md_get_stat "t_force_ms", "t_build_ms", "t_integrate_ms",
 *                    "t_other_ms", "n_force"; setting it resets the accumulators
 *   "precise_r2"     cell and neighbour-list paths: squared distance below which an in-range pair is
 *                    evaluated in FP64 from the exact cell-local coordinates.  Default 1.3 sigma^2
 *                    (1.5 sigma^2 when the cell kernel groups several cells per warp); 0 = FP32 for
 *                    every pair but the sliver around rc^2; a huge value = FP64 for every in-range
 *                    pair.  The all-pairs path always evaluates every in-range pair in FP64.
 *                    Lennard-Jones only: MD_EINVAL while another potential is set (the FP32 branch is
 *                    Lennard-Jones arithmetic; md_set_potential keeps every pair in FP64)
 *   "cell_kernel"    cell-force kernel: 2 (default) ballot filter + per-lane walk (force_cell2.cu),
 *                    1 its first version (force_cell.cu), 3 dense evaluation of every staged
 *                    candidate (force_cell3.cu); same forces within the tolerances of DESIGN.md 12
 *   "cell_order"     1 = cells numbered along a Morton curve instead of linearly (dense kernel only: selects
 *                    "cell_kernel" = 3; default 0: measured slower).  Kept across later
 *                    "skin" / "cell_skin" options.  The cell arrays are sized for n^3 ids at md_create and
 *                    enlarged to the padded cube (up to 8 n^3) only here: MD_ENOMEM if that fails,
 *                    MD_EDOMAIN without a cell grid
 *   "deterministic"  1 = MD_CELL (rebuilt every step, kernels 2 and 3): after every build each cell is re-ordered by
 *                    atom id, so forces are summed in the same order in every run and reruns are bit-identical
 *                    (the ranks inside a cell otherwise come from an atomicAdd and the last bits of a force vary
 *                    from run to run).  A debugging aid for parity failures: one more pass over the state per
 *                    step; default 0.  The all-pairs and neighbour-list paths have no such option
 *   "fuse_integrator" 1 = interior steps of md_step(MD_CELL) integrate in the force kernel's epilogue
 *                    (kernels 2 and 3; default 0: measured slower)
 *   "sort_every"     all-pairs path: re-sort atoms along the Hilbert curve every k steps (default 10)
 *   "ap_general"     1 = force the unsorted per-pair-minimum-image all-pairs kernel
 *   "ap_R"           atoms per thread (1, 2, 4, 8) of the sorted all-pairs kernel, overriding the
 *                    choice made from N and L; blocks too wide for the box test per-pair images
 *   "vl_naive_build" 1 = MD_VERLET lists built by the thread-per-atom kernel instead of the cell kernel's warp
 *                    filter (default 0; the cross-check of the two builders)
 * Any other key is MD_EINVAL.  Limits: N <= 2^30 (md_create: MD_EINVAL beyond), N <= 2^23 - 1 for MD_VERLET,
 * at most 1023 cells per dimension (a larger box gets wider cells).
 * md_get_stat keys: "ncell" (cells per dimension), "side" (cell side), "last_side" (width of the last cell of a
 * row, >= side: it takes the remainder of L), "cell_order", "cell_ids" (numbering in force and how many ids it
 * spans), "max_occupancy", "kernel_launches" (kernels launched by this handle so far, graph nodes included),
 * "graph_replays", "steps_done", "precise_r2" (the window in force),
 * "vl_builds", "vl_steps", "vl_cap", "vl_overflow" (neighbour-list builds, evaluations, capacity, and 0 or the
 * longest list any build since the last host-requested one needed beyond the capacity: sticky, so a list
 * truncated in the middle of md_step is reported at its end even if later builds fitted),
 * "ap_tiled", "ap_R", "ap_ntiles", "ap_tsplit", "ap_nsplit" (all-pairs launch shape: sorted kernel in use, atoms
 * per thread, i blocks, j splits; j splits of the general kernel), "nbr_cap" (candidate-list capacity per atom of
 * the sorted all-pairs kernel, 0 before its first use), "andersen_threshold", "andersen_steps",
 * "t_integrate_ms", "t_build_ms", "t_force_ms", "t_force2_ms", "t_other_ms", "n_force" (with "time_kernels"). */
int md_set_option(md_sim *s, const char *key, double value);
int md_get_stat(md_sim *s, const char *key, double *value);

/* Calibration helper for the benchmark, not part of the MD path: the FP32 FMA rate of the current device in
 * TFLOP/s (2 flop per FFMA), measured with a register-only kernel of independent FFMA chains at full occupancy,
 * best of three launches timed with CUDA events on cuda_stream; *ms (may be NULL) receives that launch's time.
 * bench.py reports it beside the derived "alu" peak (SMs x 128 lanes x 2 x max SM clock).  Allocates nothing. */
int md_probe_fp32_peak(double *tflops, double *ms, void *cuda_stream);

/* Text of the last CUDA error seen by this thread's library calls ("" if none). */
const char *md_last_cuda_error(void);

/* Kernels launched by rand48_fill calls so far (process-wide counter). */
int64_t rand48_kernel_launches(void);

#ifdef __cplusplus
}
#endif
#endif /* LJMD_H */
