// Cell list: per-step build as a counting sort; the force kernel (row a4)
// is in force_cell.cu.  PAPER.md:98 (cells of side >= rc), :134 (n = int[L/rc]), :112 (27 neighbour
// cells), :114-118 (the paper's serial per-cell append, replaced here by histogram + scan +
// scatter).  Cells live on a power-of-two aligned grid so that cell-local coordinates and the
// offsets between neighbouring cells are exact in FP32.
#include "common.cuh"

#define CB_T 256

__device__ __forceinline__ int cell_coord(float x, const Grid &g)
{
    int c = min((int)(x * g.inv_side), g.n - 1);
    float o = (float)c * g.side;                       // exact: a multiple of the grid quantum
    if (x < o) c--;
    else if (c < g.n - 1 && x >= o + g.side) c++;
    return c;
}

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

// Exclusive scan of cell_count -> cell_start[0..ncells], max occupancy, and reset of the
// counters for the next build.  One block; each thread owns a contiguous chunk.
__global__ void __launch_bounds__(1024)
k_scan_cells(int *__restrict__ cell_count, int *__restrict__ cell_start, int ncells, int *__restrict__ max_occ)
{
    __shared__ int wsum[32];
    __shared__ int wmax[32];
    const int t = threadIdx.x, lane = t & 31, wid = t >> 5;
    const int chunk = (ncells + 1023) / 1024;
    const int beg = min(ncells, t * chunk), end = min(ncells, beg + chunk);
    int sum = 0, mx = 0;
    for (int c = beg; c < end; c++) {
        int v = cell_count[c];
        sum += v;
        mx = max(mx, v);
    }
    int incl = sum;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
        int y = __shfl_up_sync(0xffffffffu, incl, o);
        if (lane >= o) incl += y;
    }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) mx = max(mx, __shfl_xor_sync(0xffffffffu, mx, o));
    if (lane == 31) wsum[wid] = incl;
    if (lane == 0) wmax[wid] = mx;
    __syncthreads();
    if (wid == 0) {
        int v = wsum[lane], m = wmax[lane];
        int inc2 = v;
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) {
            int y = __shfl_up_sync(0xffffffffu, inc2, o);
            if (lane >= o) inc2 += y;
        }
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) m = max(m, __shfl_xor_sync(0xffffffffu, m, o));
        wsum[lane] = inc2 - v;                 // exclusive warp offsets
        if (lane == 0) *max_occ = m;
    }
    __syncthreads();
    int run = wsum[wid] + incl - sum;          // exclusive offset of this thread's chunk
    for (int c = beg; c < end; c++) {
        int v = cell_count[c];
        cell_start[c] = run;
        cell_count[c] = 0;
        run += v;
    }
    if (t == 1023) cell_start[ncells] = run;
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

int ljmd_scan_counts(md_sim *s, int *count, int *start, int n)
{
    k_scan_cells<<<1, 1024, 0, s->stream>>>(count, start, n, s->max_occ);
    CKL(s);
    return MD_OK;
}

int ljmd_cell_build(md_sim *s)
{
    int N = (int)s->N;
    int nb = (N + CB_T - 1) / CB_T;
    k_bin<<<nb, CB_T, 0, s->stream>>>(s->pos, N, s->grid, s->cell_of, s->rank, s->cell_count);
    CKL(s);
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
