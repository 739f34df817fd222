// All-pairs O(N^2) Lennard-Jones force under minimum image.
// PAPER.md:49-52 (Eq. 1) and :70-76 (Sec. 2.1): one thread per atom i, the j atoms staged
// through shared memory in tiles shared by the block.  What differs from the paper's G80
// kernel:
//   * the inner loop is an FP32 distance FILTER: only ~0.16 % of pairs are inside rc at
//     N = 32000, so the pair term is evaluated (exactly, in FP64, from the original
//     coordinates) only for the few pairs the filter accepts;
//   * atoms are sorted into spatial tiles; a block owns one tile and stages every j tile
//     already shifted to the periodic image nearest the block's centre, so the minimum image
//     disappears from the inner loop, and r^2 - |u_i|^2 = |u_j|^2 - 2 u_i.u_j costs 3 FFMA;
//   * each thread carries R atoms i in registers (one shared-memory load feeds 3R FFMA);
//   * the j range is split across blockIdx.y so that small N still fills 148 SMs, and the
//     partial forces are combined in a deterministic second pass.
// k_force_allpairs_general is the unsorted per-pair-minimum-image variant for boxes too small
// to tile (L < ~4 rc) and the reference the tiled kernel is tested against.
#include <math.h>
#include "common.cuh"
#include "pair.cuh"

#define AP_T 128      // threads per block
#define AP_TJ 256     // j atoms staged per shared-memory tile
#define AP_RMAX 6     // atoms i per thread, at most

// ---------------------------------------------------------------------------------------
// General variant: per-pair minimum image, valid for any rc <= L/2 and any atom order.
__global__ void __launch_bounds__(AP_T)
k_force_allpairs_general(const float4 *__restrict__ pos, int N, PairParams P, float L, float invL,
                         double Ld, double invLd, int jchunk, double *__restrict__ fpart,
                         double *__restrict__ part_pe, double *__restrict__ part_w)
{
    __shared__ float4 tile[AP_T];
    __shared__ double red[32];
    const int tid = threadIdx.x;
    const int i = blockIdx.x * AP_T + tid;
    const int jbeg = blockIdx.y * jchunk;
    const int jend = min(N, jbeg + jchunk);
    const bool live = i < N;
    float4 pi = live ? pos[i] : make_float4(0.f, 0.f, 0.f, 0.f);
    double fx = 0.0, fy = 0.0, fz = 0.0, pe = 0.0, w = 0.0;

    for (int j0 = jbeg; j0 < jend; j0 += AP_T) {
        int cnt = min(AP_T, jend - j0);
        __syncthreads();
        if (tid < cnt) tile[tid] = pos[j0 + tid];
        __syncthreads();
        if (!live) continue;
#pragma unroll 4
        for (int k = 0; k < cnt; k++) {
            float4 pj = tile[k];
            float dx = pj.x - pi.x, dy = pj.y - pi.y, dz = pj.z - pi.z;
            dx = fmaf(-L, rintf(dx * invL), dx);
            dy = fmaf(-L, rintf(dy * invL), dy);
            dz = fmaf(-L, rintf(dz * invL), dz);
            float r2 = fmaf(dx, dx, fmaf(dy, dy, dz * dz));
            if (r2 < P.rc2f_filter && (j0 + k) != i) {
                // exact displacement from the stored FP32 coordinates, as the oracle sees them
                double ex = (double)pj.x - (double)pi.x;
                double ey = (double)pj.y - (double)pi.y;
                double ez = (double)pj.z - (double)pi.z;
                ex = fma(-Ld, rint(ex * invLd), ex);
                ey = fma(-Ld, rint(ey * invLd), ey);
                ez = fma(-Ld, rint(ez * invLd), ez);
                pair_f64(P, ex, ey, ez, fx, fy, fz, pe, w);
            }
        }
    }
    if (live) {
        size_t base = (size_t)blockIdx.y * 3 * N;
        fpart[base + i] = fx;
        fpart[base + (size_t)N + i] = fy;
        fpart[base + 2 * (size_t)N + i] = fz;
    }
    pe = block_sum(pe, red);
    w = block_sum(w, red);
    if (tid == 0) {
        int b = blockIdx.y * gridDim.x + blockIdx.x;
        part_pe[b] = 0.5 * pe;            // every pair is visited from both ends
        part_w[b] = 0.5 * w;
    }
}

// ---------------------------------------------------------------------------------------
// Tile sort: counting sort of the state by spatial tile (ta x tb x tc uniform boxes).
struct TileGrid { int a, b, c; float sa, sb, sc; };   // s* = count / L

__global__ void __launch_bounds__(256)
k_bin_tile(const float4 *__restrict__ pos, int N, TileGrid g, int *__restrict__ tile_of, int *__restrict__ rank,
           int *__restrict__ count)
{
    int i = blockIdx.x * 256 + threadIdx.x;
    if (i >= N) return;
    float4 p = pos[i];
    int tx = min(g.a - 1, (int)(p.x * g.sa));
    int ty = min(g.b - 1, (int)(p.y * g.sb));
    int tz = min(g.c - 1, (int)(p.z * g.sc));
    int t = (tx * g.b + ty) * g.c + tz;
    tile_of[i] = t;
    rank[i] = atomicAdd(&count[t], 1);
}

__global__ void __launch_bounds__(256)
k_scatter_tile(const float4 *__restrict__ pos, const float4 *__restrict__ vel, int N, const int *__restrict__ tile_of,
               const int *__restrict__ rank, const int *__restrict__ start, float4 *__restrict__ pos2,
               float4 *__restrict__ vel2)
{
    int i = blockIdx.x * 256 + threadIdx.x;
    if (i >= N) return;
    int dst = start[tile_of[i]] + rank[i];
    pos2[dst] = pos[i];
    vel2[dst] = vel[i];
}

// ---------------------------------------------------------------------------------------
// Exact pair term from the stored coordinates (same arithmetic as the general kernel).
__device__ __forceinline__ void ap_exact(const PairParams &P, const float4 &pi, const float4 &pj, double Ld, double invLd,
                                         double &fx, double &fy, double &fz, double &pe, double &w)
{
    double ex = (double)pj.x - (double)pi.x;
    double ey = (double)pj.y - (double)pi.y;
    double ez = (double)pj.z - (double)pi.z;
    ex = fma(-Ld, rint(ex * invLd), ex);
    ey = fma(-Ld, rint(ey * invLd), ey);
    ez = fma(-Ld, rint(ez * invLd), ez);
    pair_f64(P, ex, ey, ez, fx, fy, fz, pe, w);
}

// One block = one tile of i atoms (R per thread) against the j range [jbeg, jend).
template <int R>
__device__ __forceinline__ void ap_sweep(const float4 *__restrict__ pos, int N, const PairParams &P, float L, float invL,
                                         double Ld, double invLd, float hmax, int ibeg, int iend, int jbeg, int jend,
                                         int split, double *__restrict__ fpart, double &pe, double &w,
                                         float4 *tile, float *bb)
{
    const int tid = threadIdx.x, lane = tid & 31, wid = tid >> 5;
    int idx[R];
    float4 xi[R];
    float mn[3] = {INFINITY, INFINITY, INFINITY}, mx[3] = {-INFINITY, -INFINITY, -INFINITY};
#pragma unroll
    for (int r = 0; r < R; r++) {
        idx[r] = ibeg + tid + r * AP_T;
        if (idx[r] < iend) {
            xi[r] = pos[idx[r]];
            mn[0] = fminf(mn[0], xi[r].x); mx[0] = fmaxf(mx[0], xi[r].x);
            mn[1] = fminf(mn[1], xi[r].y); mx[1] = fmaxf(mx[1], xi[r].y);
            mn[2] = fminf(mn[2], xi[r].z); mx[2] = fmaxf(mx[2], xi[r].z);
        } else {
            idx[r] = -1;
            xi[r] = make_float4(0.f, 0.f, 0.f, 0.f);
        }
    }
    // bounding box of the block's atoms -> centre c and half extent h
#pragma unroll
    for (int d = 0; d < 3; d++) {
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) {
            mn[d] = fminf(mn[d], __shfl_xor_sync(0xffffffffu, mn[d], o));
            mx[d] = fmaxf(mx[d], __shfl_xor_sync(0xffffffffu, mx[d], o));
        }
    }
    __syncthreads();
    if (lane == 0) {
#pragma unroll
        for (int d = 0; d < 3; d++) { bb[wid * 6 + d] = mn[d]; bb[wid * 6 + 3 + d] = mx[d]; }
    }
    __syncthreads();
#pragma unroll
    for (int d = 0; d < 3; d++) {
        mn[d] = bb[d]; mx[d] = bb[3 + d];
#pragma unroll
        for (int k = 1; k < AP_T / 32; k++) {
            mn[d] = fminf(mn[d], bb[k * 6 + d]);
            mx[d] = fmaxf(mx[d], bb[k * 6 + 3 + d]);
        }
    }
    const float cx = 0.5f * (mn[0] + mx[0]), cy = 0.5f * (mn[1] + mx[1]), cz = 0.5f * (mn[2] + mx[2]);
    const float hx = 0.5f * (mx[0] - mn[0]), hy = 0.5f * (mx[1] - mn[1]), hz = 0.5f * (mx[2] - mn[2]);
    const float hm = fmaxf(hx, fmaxf(hy, hz));
    // every image chosen relative to c is the minimum image for pairs within rc iff
    // h + rc <= L/2 (with slack); otherwise fall back to per-pair minimum image
    const bool preshift = hm <= hmax;

    // filter threshold: rc^2 plus the rounding error of the 3-FFMA form at these magnitudes
    const float rcf = P.rcf;
    const float Mi = 1.7320508f * hm, M = Mi + rcf;
    const float thr = (float)P.rc2 + 2e-6f * (M * M + 2.f * M * Mi) + 8.f * rcf * (L * 1.1920929e-7f) + 1e-6f * (float)P.rc2;

    float ax[R], ay[R], az[R], T[R];
    double fx[R], fy[R], fz[R];
#pragma unroll
    for (int r = 0; r < R; r++) {
        float ux = xi[r].x - cx, uy = xi[r].y - cy, uz = xi[r].z - cz;
        ax[r] = -2.f * ux; ay[r] = -2.f * uy; az[r] = -2.f * uz;
        T[r] = (idx[r] >= 0) ? thr - fmaf(ux, ux, fmaf(uy, uy, uz * uz)) : -INFINITY;
        fx[r] = fy[r] = fz[r] = 0.0;
    }

    for (int j0 = jbeg; j0 < jend; j0 += AP_TJ) {
        __syncthreads();
        for (int t = tid; t < AP_TJ; t += AP_T) {
            int j = j0 + t;
            float4 u = make_float4(0.f, 0.f, 0.f, INFINITY);       // padding never passes the filter
            if (j < jend) {
                float4 p = pos[j];
                if (preshift) {
                    u.x = p.x - cx; u.y = p.y - cy; u.z = p.z - cz;
                    u.x = fmaf(-L, rintf(u.x * invL), u.x);
                    u.y = fmaf(-L, rintf(u.y * invL), u.y);
                    u.z = fmaf(-L, rintf(u.z * invL), u.z);
                    u.w = fmaf(u.x, u.x, fmaf(u.y, u.y, u.z * u.z));
                } else {
                    u = make_float4(p.x, p.y, p.z, 0.f);
                }
            }
            tile[t] = u;
        }
        __syncthreads();
        const int ntile = min(AP_TJ, jend - j0);
        if (preshift) {
            for (int ch = 0; ch * 32 < ntile; ch++) {
                const float4 *tj = tile + ch * 32;
                bool any[R];
#pragma unroll
                for (int r = 0; r < R; r++) any[r] = false;
#pragma unroll 8
                for (int k = 0; k < 32; k++) {
                    const float4 uj = tj[k];
#pragma unroll
                    for (int r = 0; r < R; r++) {
                        float v = fmaf(ax[r], uj.x, fmaf(ay[r], uj.y, fmaf(az[r], uj.z, uj.w)));
                        any[r] |= v < T[r];
                    }
                }
                bool anyall = false;
#pragma unroll
                for (int r = 0; r < R; r++) anyall |= any[r];
                if (__any_sync(0xffffffffu, anyall)) {
                    // rare: some lane has a candidate inside rc in this chunk of 32 j's
#pragma unroll
                    for (int r = 0; r < R; r++) {
                        if (!any[r]) continue;
                        unsigned mask = 0;
#pragma unroll 4
                        for (int k = 0; k < 32; k++) {
                            const float4 uj = tj[k];
                            float v = fmaf(ax[r], uj.x, fmaf(ay[r], uj.y, fmaf(az[r], uj.z, uj.w)));
                            mask |= (v < T[r]) ? (1u << k) : 0u;
                        }
                        while (mask) {
                            int k = __ffs(mask) - 1;
                            mask &= mask - 1;
                            int j = j0 + ch * 32 + k;
                            if (j != idx[r]) ap_exact(P, xi[r], pos[j], Ld, invLd, fx[r], fy[r], fz[r], pe, w);
                        }
                    }
                }
            }
        } else {
            // fallback for a block whose atoms are not compact: per-pair minimum image
#pragma unroll
            for (int r = 0; r < R; r++) {
                if (idx[r] < 0) continue;
                for (int k = 0; k < ntile; k++) {
                    const float4 pj = tile[k];
                    float dx = pj.x - xi[r].x, dy = pj.y - xi[r].y, dz = pj.z - xi[r].z;
                    dx = fmaf(-L, rintf(dx * invL), dx);
                    dy = fmaf(-L, rintf(dy * invL), dy);
                    dz = fmaf(-L, rintf(dz * invL), dz);
                    float r2 = fmaf(dx, dx, fmaf(dy, dy, dz * dz));
                    if (r2 < P.rc2f_filter && (j0 + k) != idx[r])
                        ap_exact(P, xi[r], pj, Ld, invLd, fx[r], fy[r], fz[r], pe, w);
                }
            }
        }
    }
    const size_t base = (size_t)split * 3 * N;
#pragma unroll
    for (int r = 0; r < R; r++) {
        if (idx[r] >= 0) {
            fpart[base + idx[r]] = fx[r];
            fpart[base + (size_t)N + idx[r]] = fy[r];
            fpart[base + 2 * (size_t)N + idx[r]] = fz[r];
        }
    }
}

__global__ void __launch_bounds__(AP_T)
k_force_allpairs_tiled(const float4 *__restrict__ pos, const int *__restrict__ tile_start, int N, PairParams P,
                       float L, float invL, double Ld, double invLd, float hmax, int jchunk,
                       double *__restrict__ fpart, double *__restrict__ part_pe, double *__restrict__ part_w)
{
    __shared__ float4 tile[AP_TJ];
    __shared__ float bb[(AP_T / 32) * 6];
    __shared__ double red[32];
    const int t = blockIdx.x, split = blockIdx.y;
    const int tb = tile_start[t], te = tile_start[t + 1];
    const int jbeg = split * jchunk, jend = min(N, jbeg + jchunk);
    double pe = 0.0, w = 0.0;
    // a tile larger than AP_T * AP_RMAX atoms takes several passes
    for (int ibeg = tb; ibeg < te; ibeg += AP_T * AP_RMAX) {
        const int iend = min(te, ibeg + AP_T * AP_RMAX);
        const int R = (iend - ibeg + AP_T - 1) / AP_T;
        switch (R) {
        case 1: ap_sweep<1>(pos, N, P, L, invL, Ld, invLd, hmax, ibeg, iend, jbeg, jend, split, fpart, pe, w, tile, bb); break;
        case 2: ap_sweep<2>(pos, N, P, L, invL, Ld, invLd, hmax, ibeg, iend, jbeg, jend, split, fpart, pe, w, tile, bb); break;
        case 3: ap_sweep<3>(pos, N, P, L, invL, Ld, invLd, hmax, ibeg, iend, jbeg, jend, split, fpart, pe, w, tile, bb); break;
        case 4: ap_sweep<4>(pos, N, P, L, invL, Ld, invLd, hmax, ibeg, iend, jbeg, jend, split, fpart, pe, w, tile, bb); break;
        case 5: ap_sweep<5>(pos, N, P, L, invL, Ld, invLd, hmax, ibeg, iend, jbeg, jend, split, fpart, pe, w, tile, bb); break;
        default: ap_sweep<6>(pos, N, P, L, invL, Ld, invLd, hmax, ibeg, iend, jbeg, jend, split, fpart, pe, w, tile, bb); break;
        }
    }
    pe = block_sum(pe, red);
    w = block_sum(w, red);
    if (threadIdx.x == 0) {
        int b = split * gridDim.x + t;
        part_pe[b] = 0.5 * pe;
        part_w[b] = 0.5 * w;
    }
}

// Deterministic combine of the j-split partial forces: frc[i] = sum_s fpart[s][.][i].
__global__ void __launch_bounds__(256)
k_combine_forces(float4 *__restrict__ frc, const double *__restrict__ fpart, int N, int nsplit)
{
    int i = blockIdx.x * 256 + threadIdx.x;
    if (i >= N) return;
    double fx = 0.0, fy = 0.0, fz = 0.0;
    for (int s = 0; s < nsplit; s++) {
        size_t base = (size_t)s * 3 * N;
        fx += fpart[base + i];
        fy += fpart[base + (size_t)N + i];
        fz += fpart[base + 2 * (size_t)N + i];
    }
    frc[i] = make_float4((float)fx, (float)fy, (float)fz, 0.0f);
}

// ---------------------------------------------------------------------------------------
// Host side: choose the tile grid (md_create), sort, launch.
void ljmd_ap_plan(md_sim *s)
{
    // tiles of ~480 atoms (R = 4 with 128 threads); every dimension needs >= amin tiles so
    // that half a tile plus rc fits in L/2
    const double L = s->L, rc = s->rc;
    const double slack = 0.05 * rc;
    s->ap_hmax = (float)(0.5 * L - rc - slack);
    s->ap_tiled = false;
    s->ap_ntiles = 0;
    double denom = L - 2.0 * (rc + slack) - 0.25;        // 0.25: atoms drift between re-sorts
    if (denom <= 0) return;
    int amin = (int)ceil(L / denom);
    if (amin < 2) amin = 2;
    const double target = 480.0;
    double best = 1e300;
    int ba = 0, bb = 0, bc = 0;
    for (int a = amin; a <= 96; a++)
        for (int b = a; b <= 96; b++)
            for (int c = b; c <= 96; c++) {
                double pop = (double)s->N / ((double)a * b * c);
                if (pop < 100.0) break;
                // prefer a population just below a multiple of AP_T (full register tiles)
                double R = ceil((pop + 3.0 * sqrt(pop) * 0.5) / AP_T);
                if (R > AP_RMAX) continue;
                double waste = 1.0 - pop / (R * AP_T) + 0.02 * fabs(pop - target) / target + 0.01 * (c - a);
                if (waste < best) { best = waste; ba = a; bb = b; bc = c; }
            }
    if (!ba) return;
    s->ap_tiled = true;
    s->ap_ta = ba; s->ap_tb = bb; s->ap_tc = bc;
    s->ap_ntiles = ba * bb * bc;
    // j splits: fill the GPU with resident blocks and balance them across the SMs
    int sms = 148;
    cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, 0);
    int maxsplit = (int)((s->N + 4 * AP_TJ - 1) / (4 * AP_TJ));     // at least 4 j tiles per block
    if (maxsplit < 1) maxsplit = 1;
    int bestsplit = 1;
    double besteff = 0.0;
    for (int k = 1; k <= maxsplit && k <= 64; k++) {
        double blocks = (double)s->ap_ntiles * k;
        double per_sm = blocks / sms;
        if (per_sm > 5.0 && k > 1) break;                            // about 5 blocks resident per SM
        double eff = per_sm / ceil(per_sm) * (per_sm >= 4.0 ? 1.0 : per_sm / 4.0);
        if (eff > besteff + 1e-9) { besteff = eff; bestsplit = k; }
    }
    s->ap_tsplit = bestsplit;
}

static int ap_tile_sort(md_sim *s)
{
    int N = (int)s->N;
    int nb = (N + 255) / 256;
    TileGrid g;
    g.a = s->ap_ta; g.b = s->ap_tb; g.c = s->ap_tc;
    g.sa = (float)(g.a / s->L); g.sb = (float)(g.b / s->L); g.sc = (float)(g.c / s->L);
    k_bin_tile<<<nb, 256, 0, s->stream>>>(s->pos, N, g, s->cell_of, s->rank, s->tile_count);
    CKL(s);
    int r = ljmd_scan_counts(s, s->tile_count, s->tile_start, s->ap_ntiles);
    if (r) return r;
    k_scatter_tile<<<nb, 256, 0, s->stream>>>(s->pos, s->vel, N, s->cell_of, s->rank, s->tile_start, s->pos2, s->vel2);
    CKL(s);
    float4 *t = s->pos; s->pos = s->pos2; s->pos2 = t;
    t = s->vel; s->vel = s->vel2; s->vel2 = t;
    return MD_OK;
}

int ljmd_forces_allpairs(md_sim *s)
{
    int N = (int)s->N;
    double *ppe = s->part + (size_t)s->part_cap;
    double *pw = s->part + 2 * (size_t)s->part_cap;
    int nsplit;
    if (s->ap_tiled && !s->ap_force_general) {
        if (s->layout != LAYOUT_TILE || s->ap_since_sort >= s->sort_every) {
            int r = ap_tile_sort(s);
            if (r) return r;
            s->layout = LAYOUT_TILE;
            s->ap_since_sort = 0;
            ljmd_tick(s, TAG_BUILD);
        }
        s->ap_since_sort++;
        nsplit = s->ap_tsplit;
        int jchunk = (N + nsplit - 1) / nsplit;
        jchunk = ((jchunk + AP_TJ - 1) / AP_TJ) * AP_TJ;
        dim3 grid(s->ap_ntiles, nsplit);
        k_force_allpairs_tiled<<<grid, AP_T, 0, s->stream>>>(s->pos, s->tile_start, N, s->pp, s->Lf, 1.0f / s->Lf,
                                                            s->L, 1.0 / s->L, s->ap_hmax, jchunk, s->fpart, ppe, pw);
        CKL(s);
        s->n_pe = s->ap_ntiles * nsplit;
    } else {
        int niblk = (N + AP_T - 1) / AP_T;
        nsplit = s->ap_nsplit;
        int jchunk = (N + nsplit - 1) / nsplit;
        jchunk = ((jchunk + AP_T - 1) / AP_T) * AP_T;
        dim3 grid(niblk, nsplit);
        k_force_allpairs_general<<<grid, AP_T, 0, s->stream>>>(s->pos, N, s->pp, s->Lf, 1.0f / s->Lf, s->L, 1.0 / s->L,
                                                              jchunk, s->fpart, ppe, pw);
        CKL(s);
        s->n_pe = niblk * nsplit;
        if (s->layout == LAYOUT_CELL) s->layout = LAYOUT_NONE;      // lpos no longer tracked
    }
    ljmd_tick(s, TAG_FORCE);
    k_combine_forces<<<(N + 255) / 256, 256, 0, s->stream>>>(s->frc, s->fpart, N, nsplit);
    CKL(s);
    ljmd_tick(s, TAG_OTHER);
    return MD_OK;
}
