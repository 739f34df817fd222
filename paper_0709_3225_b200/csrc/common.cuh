// Internal declarations shared by the translation units of libljmd_b200.so.
// Public surface: include/ljmd.h.  Nothing here is shared with oracle/.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>
#include "../../include/ljmd.h"

#define LJ_WARP 32

// ---- error plumbing -------------------------------------------------------------
void ljmd_note_cuda_error(cudaError_t e, const char *what, const char *file, int line);
#define CK(call)                                                        \
    do {                                                                \
        cudaError_t e__ = (call);                                       \
        if (e__ != cudaSuccess) {                                       \
            ljmd_note_cuda_error(e__, #call, __FILE__, __LINE__);       \
            return MD_ECUDA;                                            \
        }                                                               \
    } while (0)
#define CKL(s) CK(cudaGetLastError()); (s)->launches++

// ---- device memory (through the optional allocator hooks) -----------------------
void *ljmd_dev_alloc(int64_t bytes, cudaStream_t st);
void ljmd_dev_free(void *p, cudaStream_t st);

// ---- pair-potential constants, FP64 (precise branch) and FP32 (filters, fast branch)
struct PairParams {
    double rc2, sig2, eps24, eps4, ushift, rc, f_rc;   // f_rc = f_LJ(rc), mode 2 only
    double precise_r2;     // pairs with r2 < precise_r2 are evaluated in FP64
    float rc2f_filter;     // FP32 accept threshold (rc^2 plus a rounding margin)
    float sig2f, eps24f, eps4f, ushiftf, rcf, f_rcf;
    int mode;
    int kind;              // MD_POT_LJ or MD_POT_YUKAWA (md_set_potential)
    double yA, ykappa;     // Yukawa: U = yA exp(-ykappa r) / r
};

// ---- cell grid on a power-of-two aligned lattice ----------
struct Grid {
    int n;            // cells per dimension
    int ncells;       // n^3
    float side;       // width of cells 0..n-2 (a multiple of the grid quantum g)
    float last;       // width of cell n-1 = L - (n-1)*side  (>= side)
    float inv_side;
    float L;
    int morton;       // option "cell_order" = 1 (dense kernel only): cells numbered along a Morton curve
    int nid;          // number of cell ids: n^3, or P^3 with P = the power of two >= n for the Morton numbering
};

// One cached graph: valid for this force path and exactly this host-side state at the unit's start
#define MD_NGRAPH 4
struct GraphEntry {
    cudaGraphExec_t exec;
    int algo, unit, since_sort, layout, stamp;
    void *pos, *vel, *lpos;
    int64_t launches;             // kernels per replay
    cudaStream_t stream;
};

// Control block of k_scan_cells (device memory; cells.cu)
struct ScanCtl {
    unsigned ticket;              // monotonic block ticket counter
    unsigned base;                // ticket of tile 0 of the current launch
    unsigned done;                // blocks of the current launch that have finished
    unsigned pad;
    unsigned long long epoch;     // launch number (30 bits), tags the look-back words and max_occ
};

// Device-side control block of the neighbour-list path (verlet.cu)
struct VlCtl {
    unsigned maxd2;               // bits of the largest squared displacement since the last build
    int rebuild;                  // this step's decision (read by the build kernels)
    int force;                    // host request: build at the next evaluation
    int overflow;                 // 0, or the longest list length the last build needed when it exceeded the capacity
    int nbuilds, nsteps;          // statistics
};

enum { TAG_START = -1, TAG_INTEGRATE = 0, TAG_BUILD = 1, TAG_FORCE = 2, TAG_OTHER = 3, TAG_FORCE2 = 4, TAG_COUNT = 5 };

struct md_sim {
    int64_t N;
    double L, rc, eps, sigma, dt;
    int shifted;
    int pot_kind;         // md_set_potential
    double pot_a, pot_b;
    float Lf, dtf, hdtf;
    PairParams pp;
    Grid grid;            // grid.n == 0 when the box has fewer than 3 cells per dimension
    Grid vgrid;           // cells of side >= rc + skin for the neighbour-list path (n == 0: unavailable)
    double skin;
    unsigned *vl_list;    // [vl_cap][vl_npad] slot of j | offset index << 23
    int *vl_count;        // [N]
    float4 *vl_lbuild;    // [N] local coordinates at the last build
    VlCtl *vl_ctl;
    int vl_cap, vl_npad;
    bool vl_fuse;         // option "vl_fuse": interior steps of md_step(MD_VERLET) integrate in the force kernel's epilogue
    bool vl_half;         // option "vl_half": half lists + vector reductions for the reactions (measurement)
    bool vl_naive_build;  // option "vl_naive_build": thread-per-atom list kernel instead of the warp filter
    int grid_paper_n;     // int[L/rc]
    cudaStream_t stream;

    // state in "slot" order; pos.w carries the caller's atom id as int bits
    float4 *pos, *vel, *frc;
    float4 *pos2, *vel2;          // scatter targets (cell build)
    float4 *lpos;                 // cell-local coordinates in slot order (after a build)
    float4 *lpos2;                // list path with the fused integrator: the local coordinates of the next step
    int *cell_of;                 // [N] cell id per slot (after a build)
    int *rank;                    // [N] rank inside its cell (during a build)
    int *cell_count;              // [ncells]
    int *cell_start;              // [ncells + 1]
    unsigned long long *max_occ;  // [1] epoch << 32 | max cell occupancy of the last scan
    // multi-block scan: device-side control block and per-tile look-back words
    ScanCtl *scan_ctl;
    unsigned long long *scan_state;
    int scan_cap;
    // all-pairs partial forces: [nsplit][3][N] doubles
    double *fpart;
    int ap_nsplit;                // j splits of the general kernel
    unsigned *ap_tile_done;       // [i blocks] arrival counters of the general kernel (zero between launches)
    // all-pairs tiled kernel: R atoms per thread, i blocks, j splits, Morton sort grid,
    // pre-shift validity bound
    bool ap_tiled, ap_force_general;
    int ap_R, ap_ntiles, ap_tsplit, ap_since_sort, ap_sort_g, ap_sort_bins;
    float ap_hmax;
    int *tile_count, *tile_start;
    // candidate lists of the sorted all-pairs kernel (allocated on first use)
    int *nbr_count, *nbr_list;    // [N], [N][nbr_cap]
    int nbr_cap;
    // energy partials and results
    double *part;                 // [3][part_cap] block partials: KE, PE, W
    int part_cap;
    int n_ke, n_pe;               // valid partial counts
    double *energies;             // [3] on device: KE, PE, W
    float *xfer;                  // [N][3] staging for host/device packing
    int layout;                   // LAYOUT_*: how the slots are currently ordered
    bool has_state, forces_valid;
    bool binned;                  // cell_of/rank/cell_count already hold the histogram of the current positions
    bool binned3;                 // lean build: vel.w/cell_count hold the histogram of the current positions
    bool fused_pending;           // the last force kernel integrated: pos2 = drifted positions, vel = kicked velocities with ranks in .w
    int forces_algo;
    bool use_graph;
    int sort_every;
    // Andersen thermostat (options "andersen_nu", "andersen_T", "andersen_seed"); and_thr = 0: off
    uint32_t and_thr;
    double and_T, and_nu;
    uint64_t and_seed, and_t;     // stream start state, steps since it was (re)configured
    uint64_t *and_t_dev;          // the same count in device memory (read by the thermostat kernel, graph-replayable)
    bool precise_r2_user;         // "precise_r2" was set through md_set_option
    int cell_group;               // cells per row group of the cell-force kernel; 0 = automatic
    int cell_kernel;              // 2 (default): force_cell2.cu; 3: force_cell3.cu (dense); 1: force_cell.cu
    bool deterministic;           // option "deterministic": cells re-ordered by atom id after every build (cells.cu)
    float4 *lpos_det;             // twin of lpos for that pass (allocated when the option is switched on)
    int cell_order;               // option "cell_order" (1 = Morton numbering); re-applied to `grid` whenever it is rebuilt
    int cell_cap;                 // ints allocated for cell_count (cell_start has one more)
    bool cell_skin_on;            // option "cell_skin" > 0: MD_CELL runs on skin cells (verlet.cu)
    bool fuse_integrator;         // option "fuse_integrator": interior steps integrate in the force kernel's epilogue
    int64_t launches, steps_done;
    // CUDA graphs of one "unit" of interior steps (ljmd_api.cu): the unit is the number of steps after
    // which the host-side state (buffer roles, re-sort phase) repeats, so the graph can be replayed
    GraphEntry graphs[MD_NGRAPH];
    int graph_clock;              // LRU stamp
    cudaStream_t cap_stream;      // capture/replay stream when the caller's stream is the legacy default
    int64_t graph_replays;
    // optional per-phase timing with CUDA events on s->stream ("time_kernels" option)
    bool time_kernels;
    cudaEvent_t *ev_pool;
    int *ev_tag;
    int ev_cap, ev_n;
    double t_phase[TAG_COUNT];    // ms: integrate, build, force kernel, other, second force kernel
    int64_t n_phase[TAG_COUNT];
};

enum { LAYOUT_NONE = 0, LAYOUT_CELL = 1, LAYOUT_TILE = 2, LAYOUT_VERLET = 3, LAYOUT_SKINCELL = 4 };
// Record an event; the time since the previous tick is attributed to `tag`.
void ljmd_tick(md_sim *s, int tag);
int ljmd_collect_ticks(md_sim *s);
void ljmd_drop_graphs(md_sim *s);                   // ljmd_api.cu: forget every cached CUDA graph of the handle

// ---- kernels' host launchers (each returns md_status) ---------------------------
int ljmd_pack_state(md_sim *s, const float *dpos, const float *dvel);
int ljmd_unpack(md_sim *s, const float4 *src, float *dout);        // [N][3], caller's order
int ljmd_kick_drift(md_sim *s, int kicks);           // kicks = 2: plus the pending half-kick of the previous step
int ljmd_kick_drift_bin(md_sim *s, int kicks);       // same, fused with the cell histogram
int ljmd_kick_ke(md_sim *s);
int ljmd_ke_only(md_sim *s);
int ljmd_reduce_energies(md_sim *s);
int ljmd_forces_allpairs(md_sim *s);
void ljmd_ap_plan(md_sim *s);
void ljmd_ap_set_R(md_sim *s, int R);                       // R in {0 (general kernel), 1, 2, 4, 8}
int ljmd_scan_counts(md_sim *s, int *count, int *start, int n, const int *cond = nullptr);   // exclusive scan, zeroes count; cond: device flag, 0 = do nothing
int ljmd_kick_andersen(md_sim *s);                   // rand48.cu: second half-kick + thermostat + KE
int ljmd_mb_velocities(md_sim *s, double T, uint64_t seed48, double *vraw, double *part, double *mom);   // rand48.cu
int ljmd_vl_kick_drift(md_sim *s, int kicks);
int ljmd_vl_build_lists(md_sim *s, const int *cond);    // force_cell.cu: lists through the cell kernel's filter
int ljmd_forces_verlet(md_sim *s, bool fuse = false);   // fuse: the epilogue integrates (full lists)
int ljmd_vl_stats(md_sim *s, int *nbuilds, int *nsteps, int *overflow);
int ljmd_vl_grow(md_sim *s, int need);               // longer lists after an overflow; the next evaluation rebuilds
int ljmd_cell_build(md_sim *s);
int ljmd_forces_cell(md_sim *s);
int ljmd_forces_cell2_on(md_sim *s, const Grid &g, double stray, bool energy, bool fused);   // the same on any grid whose lpos/cell_start are current
int ljmd_forces_skincell(md_sim *s, bool energy);    // verlet.cu: cells of side >= rc + skin, re-sorted when the skin is used up
int ljmd_forces_cell2(md_sim *s, bool energy, bool fused);   // force_cell2.cu; energy = false: forces only; fused: the epilogue integrates
int ljmd_forces_cell3(md_sim *s, bool energy, bool fused);   // force_cell3.cu; fused: the epilogue integrates
int ljmd_kick_drift_bin3(md_sim *s, int kicks);      // cells.cu: lean build (rank in vel.w)
int ljmd_cell_build3(md_sim *s);

// ---- small device helpers --------------------------------------------------------
// Wrap x into [0,L) after a drift of less than L (R14): a result that rounds to L becomes 0.
__device__ __forceinline__ float wrap_drift(float x, float L)
{
    if (x >= L) x -= L;
    else if (x < 0.0f) x += L;
    if (x >= L || x < 0.0f) x = 0.0f;
    return x;
}

// Cell index of coordinate x in [0,L) (cells 0..n-2 of width side, the last one takes the remainder):
// the reciprocal multiply is corrected against the exact cell origins.
__device__ __forceinline__ int cell_coord(float x, const Grid &g)
{
    int c = min((int)(x * g.inv_side), g.n - 1);
    float o = (float)c * g.side;                       // exact: a multiple of the grid quantum
    if (x < o) c--;
    else if (c < g.n - 1 && x >= o + g.side) c++;
    return c;
}

// Cell number of cell (cx, cy, cz): linear (a z-column is one contiguous run of slots), or along a Morton curve
// (north_star (b): "optional Morton or linear cell ordering"; ids of the padded cube P^3, unused ids stay empty).
__host__ __device__ __forceinline__ unsigned morton_spread(unsigned v)
{
    v &= 0x3ffu;
    v = (v | (v << 16)) & 0x030000ffu;
    v = (v | (v << 8)) & 0x0300f00fu;
    v = (v | (v << 4)) & 0x030c30c3u;
    v = (v | (v << 2)) & 0x09249249u;
    return v;
}

__host__ __device__ __forceinline__ unsigned morton_compact(unsigned v)
{
    v &= 0x09249249u;
    v = (v | (v >> 2)) & 0x030c30c3u;
    v = (v | (v >> 4)) & 0x0300f00fu;
    v = (v | (v >> 8)) & 0x030000ffu;
    v = (v | (v >> 16)) & 0x3ffu;
    return v;
}

__device__ __forceinline__ int cell_id(int cx, int cy, int cz, const Grid &g)
{
    if (g.morton) return (int)((morton_spread((unsigned)cx) << 2) | (morton_spread((unsigned)cy) << 1) | morton_spread((unsigned)cz));
    return (cx * g.n + cy) * g.n + cz;
}

__device__ __forceinline__ double warp_sum(double v)
{
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
    return v;
}

// Sum over the block; result valid in thread 0.  blockDim.x a multiple of 32, <= 1024.
__device__ __forceinline__ double block_sum(double v, double *smem32)
{
    v = warp_sum(v);
    int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
    __syncthreads();
    if (lane == 0) smem32[w] = v;
    __syncthreads();
    int nw = (blockDim.x + 31) >> 5;
    v = (threadIdx.x < nw) ? smem32[threadIdx.x] : 0.0;
    if (w == 0) v = warp_sum(v);
    return v;
}
