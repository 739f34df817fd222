// Cell list: per-step build as a counting sort; the force kernel (row a4)
// is in force_cell.cu.  PAPER.md:98 (cells of side >= rc), :134 (n = int[L/rc]), :112 (27 neighbour
// cells), :114-118 (the paper's serial per-cell append, replaced here by histogram + scan +
// scatter).  Cells live on a power-of-two aligned grid so that cell-local coordinates and the
// offsets between neighbouring cells are exact in FP32.
#include "common.cuh"

#define CB_T 256

// Histogram with the rank inside the cell returned by the atomic.
__global__ void __launch_bounds__(CB_T)
k_bin(const float4 *__restrict__ pos, int N, Grid g, int *__restrict__ cell_of, int *__restrict__ rank,
      int *__restrict__ cell_count)
{
    int i = blockIdx.x * CB_T + threadIdx.x;
    if (i >= N) return;
    float4 p = pos[i];
    int c = (cell_coord(p.x, g) * g.n + cell_coord(p.y, g)) * g.n + cell_coord(p.z, g);
    cell_of[i] = c;
    rank[i] = atomicAdd(&cell_count[c], 1);
}

// a1 + first half of a3 in one pass: [pending half-kick,] half-kick, drift, wrap, then the
// histogram of the new position.  Same arithmetic as k_kick_drift (integrate.cu).
template <int KICKS>
__global__ void __launch_bounds__(CB_T)
k_kick_drift_bin(float4 *__restrict__ pos, float4 *__restrict__ vel, const float4 *__restrict__ frc, int N,
                 float hdt, float dt, Grid g, int *__restrict__ cell_of, int *__restrict__ rank,
                 int *__restrict__ cell_count)
{
    int i = blockIdx.x * CB_T + threadIdx.x;
    if (i >= N) return;
    float4 p = pos[i], v = vel[i];
    const float4 f = frc[i];
#pragma unroll
    for (int k = 0; k < KICKS; k++) {
        v.x = fmaf(hdt, f.x, v.x);
        v.y = fmaf(hdt, f.y, v.y);
        v.z = fmaf(hdt, f.z, v.z);
    }
    p.x = wrap_drift(fmaf(dt, v.x, p.x), g.L);
    p.y = wrap_drift(fmaf(dt, v.y, p.y), g.L);
    p.z = wrap_drift(fmaf(dt, v.z, p.z), g.L);
    pos[i] = p;
    vel[i] = v;
    int c = (cell_coord(p.x, g) * g.n + cell_coord(p.y, g)) * g.n + cell_coord(p.z, g);
    cell_of[i] = c;
    rank[i] = atomicAdd(&cell_count[c], 1);
}

// Exclusive scan of cell_count -> cell_start[0..ncells], max occupancy, and reset of the
// counters for the next build.  Single pass over any number of cells: blocks take tiles of
// SC_TILE cells in ticket order and chain their prefixes through `state` with a decoupled
// look-back (one 64-bit word per tile: value | kind << 32 | epoch << 34, so words of earlier
// launches read as "empty" and nothing has to be cleared between launches).  The ticket base and
// the epoch live in device memory and are advanced by the last block to finish, so the launch has
// no per-call host arguments and can be replayed from a CUDA graph.
#define SC_T 256
#define SC_ITEMS 8
#define SC_TILE (SC_T * SC_ITEMS)
#define SC_AGG 1ull
#define SC_PREFIX 2ull

__device__ __forceinline__ unsigned long long sc_word(unsigned long long epoch, unsigned long long kind, int v)
{
    return (epoch << 34) | (kind << 32) | (unsigned)v;
}

__global__ void __launch_bounds__(SC_T)
k_scan_cells(int *__restrict__ cell_count, int *__restrict__ cell_start, int ncells,
             unsigned long long *__restrict__ max_occ, ScanCtl *__restrict__ ctl,
             volatile unsigned long long *__restrict__ state, const int *__restrict__ cond)
{
    if (cond && !*cond) return;                                // conditional launch (verlet.cu): nothing is touched
    __shared__ int wsum[SC_T / 32];
    __shared__ int s_tile, s_prefix;
    __shared__ unsigned s_base;
    __shared__ unsigned long long s_epoch;
    const int t = threadIdx.x, lane = t & 31, wid = t >> 5;
    if (t == 0) {
        s_base = *(volatile unsigned *)&ctl->base;             // stable while any block of this launch runs
        s_epoch = *(volatile unsigned long long *)&ctl->epoch;
        s_tile = (int)(atomicAdd(&ctl->ticket, 1u) - s_base);
    }
    __syncthreads();
    const int tile = s_tile;
    const unsigned long long epoch = s_epoch;
    const int base = tile * SC_TILE + t * SC_ITEMS;      // SC_ITEMS consecutive cells per thread
    int v[SC_ITEMS];
    int sum = 0, mx = 0;
    if (base + SC_ITEMS <= ncells) {
        const int4 a = *reinterpret_cast<const int4 *>(cell_count + base);
        const int4 b = *reinterpret_cast<const int4 *>(cell_count + base + 4);
        v[0] = a.x; v[1] = a.y; v[2] = a.z; v[3] = a.w; v[4] = b.x; v[5] = b.y; v[6] = b.z; v[7] = b.w;
    } else {
#pragma unroll
        for (int k = 0; k < SC_ITEMS; k++) v[k] = (base + k < ncells) ? cell_count[base + k] : 0;
    }
#pragma unroll
    for (int k = 0; k < SC_ITEMS; k++) { sum += v[k]; mx = max(mx, v[k]); }
    int incl = sum;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
        int y = __shfl_up_sync(0xffffffffu, incl, o);
        if (lane >= o) incl += y;
    }
    mx = __reduce_max_sync(0xffffffffu, mx);
    if (lane == 31) wsum[wid] = incl;
    // epoch-tagged maximum: a later launch always wins, so the word is never reset
    if (lane == 0) atomicMax(max_occ, (epoch << 32) | (unsigned)mx);
    __syncthreads();
    if (wid == 0) {
        int ws = (lane < SC_T / 32) ? wsum[lane] : 0;
        int inc2 = ws;
#pragma unroll
        for (int o = 1; o < SC_T / 32; o <<= 1) {
            int y = __shfl_up_sync(0xffffffffu, inc2, o);
            if (lane >= o) inc2 += y;
        }
        const int agg = __shfl_sync(0xffffffffu, inc2, SC_T / 32 - 1);
        if (lane < SC_T / 32) wsum[lane] = inc2 - ws;          // exclusive warp offsets
        // publish the tile aggregate, then look back for the exclusive prefix
        int prefix = 0;
        if (tile == 0) {
            if (lane == 0) state[0] = sc_word(epoch, SC_PREFIX, agg);
        } else {
            if (lane == 0) state[tile] = sc_word(epoch, SC_AGG, agg);
            int look = tile - 1;
            for (;;) {
                const int idx = look - lane;
                unsigned long long w = 0;
                bool ready;
                do {
                    w = (idx >= 0) ? state[idx] : sc_word(epoch, SC_PREFIX, 0);
                    ready = (w >> 34) == epoch && ((w >> 32) & 3ull) != 0ull;
                } while (!__all_sync(0xffffffffu, ready));
                const bool is_p = ((w >> 32) & 3ull) == SC_PREFIX;
                const unsigned pm = __ballot_sync(0xffffffffu, is_p);
                const int first_p = pm ? (__ffs(pm) - 1) : 32;          // nearest tile with a full prefix
                int val = (lane <= first_p) ? (int)(unsigned)(w & 0xffffffffull) : 0;
                prefix += __reduce_add_sync(0xffffffffu, val);
                if (pm) break;
                look -= 32;
            }
            if (lane == 0) {
                __threadfence();
                state[tile] = sc_word(epoch, SC_PREFIX, prefix + agg);
            }
        }
        if (lane == 0) s_prefix = prefix;
    }
    __syncthreads();
    int run = s_prefix + wsum[wid] + incl - sum;          // exclusive offset of this thread's first cell
    int o[SC_ITEMS];
#pragma unroll
    for (int k = 0; k < SC_ITEMS; k++) { o[k] = run; run += v[k]; }
    if (base + SC_ITEMS <= ncells) {
        *reinterpret_cast<int4 *>(cell_start + base) = make_int4(o[0], o[1], o[2], o[3]);
        *reinterpret_cast<int4 *>(cell_start + base + 4) = make_int4(o[4], o[5], o[6], o[7]);
        *reinterpret_cast<int4 *>(cell_count + base) = make_int4(0, 0, 0, 0);
        *reinterpret_cast<int4 *>(cell_count + base + 4) = make_int4(0, 0, 0, 0);
        if (base + SC_ITEMS == ncells) cell_start[ncells] = run;
    } else {
#pragma unroll
        for (int k = 0; k < SC_ITEMS; k++)
            if (base + k < ncells) { cell_start[base + k] = o[k]; cell_count[base + k] = 0; }
        if (base < ncells) cell_start[ncells] = run;      // the thread holding the last cell
    }
    // the last block to finish opens the next launch: new ticket base, next epoch
    __syncthreads();
    if (t == 0) {
        __threadfence();
        if (atomicAdd(&ctl->done, 1u) == gridDim.x - 1) {
            ctl->done = 0u;
            ctl->base = s_base + gridDim.x;
            const unsigned long long e1 = (epoch + 1ull) & 0x3fffffffull;
            ctl->epoch = e1 ? e1 : 1ull;                               // 0 marks never-written words
            __threadfence();
        }
    }
}

// Scatter into cell order: state (global coordinates) and cell-local coordinates.
__global__ void __launch_bounds__(CB_T)
k_scatter(const float4 *__restrict__ pos, const float4 *__restrict__ vel, int N, Grid g,
          const int *__restrict__ cell_of, const int *__restrict__ rank, const int *__restrict__ cell_start,
          float4 *__restrict__ pos2, float4 *__restrict__ vel2, float4 *__restrict__ lpos)
{
    int i = blockIdx.x * CB_T + threadIdx.x;
    if (i >= N) return;
    int c = cell_of[i];
    int dst = cell_start[c] + rank[i];
    float4 p = pos[i];
    int cz = c % g.n, cy = (c / g.n) % g.n, cx = c / (g.n * g.n);
    float4 l;
    l.x = p.x - (float)cx * g.side;                    // exact
    l.y = p.y - (float)cy * g.side;
    l.z = p.z - (float)cz * g.side;
    l.w = __int_as_float(c);
    pos2[dst] = p;
    vel2[dst] = vel[i];
    lpos[dst] = l;
}

int ljmd_scan_counts(md_sim *s, int *count, int *start, int n, const int *cond)
{
    const int nb = (n + SC_TILE - 1) / SC_TILE;
    if (nb > s->scan_cap) return MD_ENOMEM;
    k_scan_cells<<<nb, SC_T, 0, s->stream>>>(count, start, n, s->max_occ, s->scan_ctl, s->scan_state, cond);
    CKL(s);
    return MD_OK;
}

int ljmd_kick_drift_bin(md_sim *s, int kicks)
{
    int N = (int)s->N;
    int nb = (N + CB_T - 1) / CB_T;
    if (kicks == 2)
        k_kick_drift_bin<2><<<nb, CB_T, 0, s->stream>>>(s->pos, s->vel, s->frc, N, s->hdtf, s->dtf, s->grid, s->cell_of,
                                                        s->rank, s->cell_count);
    else
        k_kick_drift_bin<1><<<nb, CB_T, 0, s->stream>>>(s->pos, s->vel, s->frc, N, s->hdtf, s->dtf, s->grid, s->cell_of,
                                                        s->rank, s->cell_count);
    CKL(s);
    s->binned = true;
    return MD_OK;
}

int ljmd_cell_build(md_sim *s)
{
    int N = (int)s->N;
    int nb = (N + CB_T - 1) / CB_T;
    if (!s->binned) {
        k_bin<<<nb, CB_T, 0, s->stream>>>(s->pos, N, s->grid, s->cell_of, s->rank, s->cell_count);
        CKL(s);
    }
    s->binned = false;
    int r = ljmd_scan_counts(s, s->cell_count, s->cell_start, s->grid.ncells);
    if (r) return r;
    k_scatter<<<nb, CB_T, 0, s->stream>>>(s->pos, s->vel, N, s->grid, s->cell_of, s->rank, s->cell_start,
                                         s->pos2, s->vel2, s->lpos);
    CKL(s);
    float4 *t = s->pos; s->pos = s->pos2; s->pos2 = t;
    t = s->vel; s->vel = s->vel2; s->vel2 = t;
    s->layout = LAYOUT_CELL;
    return MD_OK;
}

// ---- lean build (force_cell2.cu, force_cell3.cu): the rank returned by the histogram's atomic rides in vel.w,
// the scatter recomputes the cell from the position: no cell_of/rank arrays (16 B/atom less traffic), and the
// histogram can ride in the epilogue of the force kernel (option "fuse_integrator").
__global__ void __launch_bounds__(CB_T)
k_bin3(const float4 *__restrict__ pos, float4 *__restrict__ vel, int N, Grid g, int *__restrict__ cell_count)
{
    int i = blockIdx.x * CB_T + threadIdx.x;
    if (i >= N) return;
    const float4 p = pos[i];
    const int c = cell_id(cell_coord(p.x, g), cell_coord(p.y, g), cell_coord(p.z, g), g);
    reinterpret_cast<int *>(vel)[4 * i + 3] = atomicAdd(&cell_count[c], 1);
}

template <int KICKS>
__global__ void __launch_bounds__(CB_T)
k_kick_drift_bin3(float4 *__restrict__ pos, float4 *__restrict__ vel, const float4 *__restrict__ frc, int N,
                  float hdt, float dt, Grid g, int *__restrict__ cell_count)
{
    int i = blockIdx.x * CB_T + threadIdx.x;
    if (i >= N) return;
    float4 p = pos[i], v = vel[i];
    const float4 f = frc[i];
#pragma unroll
    for (int k = 0; k < KICKS; k++) {
        v.x = fmaf(hdt, f.x, v.x);
        v.y = fmaf(hdt, f.y, v.y);
        v.z = fmaf(hdt, f.z, v.z);
    }
    p.x = wrap_drift(fmaf(dt, v.x, p.x), g.L);
    p.y = wrap_drift(fmaf(dt, v.y, p.y), g.L);
    p.z = wrap_drift(fmaf(dt, v.z, p.z), g.L);
    const int c = cell_id(cell_coord(p.x, g), cell_coord(p.y, g), cell_coord(p.z, g), g);
    v.w = __int_as_float(atomicAdd(&cell_count[c], 1));
    pos[i] = p;
    vel[i] = v;
}

__global__ void __launch_bounds__(CB_T)
k_scatter3(const float4 *__restrict__ pos, const float4 *__restrict__ vel, int N, Grid g,
           const int *__restrict__ cell_start, float4 *__restrict__ pos2, float4 *__restrict__ vel2,
           float4 *__restrict__ lpos)
{
    int i = blockIdx.x * CB_T + threadIdx.x;
    if (i >= N) return;
    const float4 p = pos[i];
    float4 v = vel[i];
    const int c = cell_id(cell_coord(p.x, g), cell_coord(p.y, g), cell_coord(p.z, g), g);
    const int dst = cell_start[c] + __float_as_int(v.w);
    v.w = 0.f;
    pos2[dst] = p;
    vel2[dst] = v;
    if (lpos) {                                        // cell-local copy for the filter kernels (force_cell2.cu); linear ids
        const int cz = c % g.n, cy = (c / g.n) % g.n, cx = c / (g.n * g.n);
        lpos[dst] = make_float4(p.x - (float)cx * g.side, p.y - (float)cy * g.side, p.z - (float)cz * g.side,
                                __int_as_float(c));    // exact
    }
}

// Option "deterministic": the rank of an atom inside its cell comes from an atomicAdd, so the slot order inside a
// cell -- and with it the order in which a force is summed, i.e. its last bits -- differs from run to run.  This
// pass re-orders every cell by the caller's atom id (carried in pos.w): rank = number of atoms of the same cell with
// a smaller id, O(occupancy^2) reads per cell out of L1/L2.  A debugging aid (bit-identical reruns), off by default.
__global__ void __launch_bounds__(CB_T)
k_order_cells(const float4 *__restrict__ pos, const float4 *__restrict__ vel, const float4 *__restrict__ lpos, int N, Grid g,
              const int *__restrict__ cell_start, float4 *__restrict__ pos2, float4 *__restrict__ vel2,
              float4 *__restrict__ lpos2)
{
    int i = blockIdx.x * CB_T + threadIdx.x;
    if (i >= N) return;
    const float4 p = pos[i];
    const int c = cell_id(cell_coord(p.x, g), cell_coord(p.y, g), cell_coord(p.z, g), g);
    const int beg = cell_start[c], end = cell_start[c + 1];
    const int id = __float_as_int(p.w);
    int rank = 0;
    for (int j = beg; j < end; j++) rank += (__float_as_int(pos[j].w) < id) ? 1 : 0;
    const int dst = beg + rank;
    pos2[dst] = p;
    vel2[dst] = vel[i];
    if (lpos) lpos2[dst] = lpos[i];
}

int ljmd_kick_drift_bin3(md_sim *s, int kicks)
{
    int N = (int)s->N;
    int nb = (N + CB_T - 1) / CB_T;
    if (kicks == 2)
        k_kick_drift_bin3<2><<<nb, CB_T, 0, s->stream>>>(s->pos, s->vel, s->frc, N, s->hdtf, s->dtf, s->grid, s->cell_count);
    else
        k_kick_drift_bin3<1><<<nb, CB_T, 0, s->stream>>>(s->pos, s->vel, s->frc, N, s->hdtf, s->dtf, s->grid, s->cell_count);
    CKL(s);
    s->binned3 = true;
    return MD_OK;
}

// Scan + scatter.  After a fused force kernel (s->fused_pending) the drifted positions are in pos2 and the
// kicked velocities (with ranks) in vel; otherwise pos/vel hold the state, histogrammed or not.
int ljmd_cell_build3(md_sim *s)
{
    int N = (int)s->N;
    int nb = (N + CB_T - 1) / CB_T;
    const bool pending = s->fused_pending;
    float4 *lp = (s->cell_kernel == 3) ? nullptr : s->lpos;      // the dense kernel reads the positions as stored
    if (!pending && !s->binned3) {
        k_bin3<<<nb, CB_T, 0, s->stream>>>(s->pos, s->vel, N, s->grid, s->cell_count);
        CKL(s);
    }
    s->binned3 = false;
    s->fused_pending = false;
    int r = ljmd_scan_counts(s, s->cell_count, s->cell_start, s->grid.nid);
    if (r) return r;
    if (pending) {
        k_scatter3<<<nb, CB_T, 0, s->stream>>>(s->pos2, s->vel, N, s->grid, s->cell_start, s->pos, s->vel2, lp);
        CKL(s);
    } else {
        k_scatter3<<<nb, CB_T, 0, s->stream>>>(s->pos, s->vel, N, s->grid, s->cell_start, s->pos2, s->vel2, lp);
        CKL(s);
        float4 *t = s->pos; s->pos = s->pos2; s->pos2 = t;
    }
    float4 *t = s->vel; s->vel = s->vel2; s->vel2 = t;
    if (s->deterministic) {
        // pos2 and vel2 are free now (they held the pre-scatter state); the cell-local copies go to their twin
        k_order_cells<<<nb, CB_T, 0, s->stream>>>(s->pos, s->vel, lp, N, s->grid, s->cell_start, s->pos2, s->vel2,
                                                  lp ? s->lpos_det : nullptr);
        CKL(s);
        t = s->pos; s->pos = s->pos2; s->pos2 = t;
        t = s->vel; s->vel = s->vel2; s->vel2 = t;
        if (lp) { t = s->lpos; s->lpos = s->lpos_det; s->lpos_det = t; }
    }
    s->layout = LAYOUT_CELL;
    return MD_OK;
}
