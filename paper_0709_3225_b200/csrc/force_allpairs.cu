// All-pairs O(N^2) Lennard-Jones force under minimum image.
// PAPER.md:49-52 (Eq. 1) and :70-76 (Sec. 2.1): one thread per atom i, the j atoms staged
// through shared memory in tiles shared by the block.  Every one of the N^2 ordered pair
// distances is computed; what differs from the paper's G80 kernel:
//   * the inner loop is an FP32 distance FILTER in 3 FFMA per pair: atoms are sorted along a
//     Hilbert curve, a block (one warp) owns 32 R consecutive atoms, and every chunk of 32 j atoms is
//     staged (per warp, no block barrier) already shifted to the periodic image nearest the
//     block's centre c, so the minimum image leaves the inner loop and
//     r^2 - |u_i|^2 = |u_j|^2 - 2 u_i.u_j  (u = x - c);
//   * the cutoff test is folded into a running minimum (one FMNMX3 per two pairs); only a
//     32-j chunk whose minimum drops below the threshold is rescanned into hit masks;
//   * the hits (0.16 % of the pairs at N = 32000) are appended to per-atom lists in global
//     memory (one atomic per non-empty 32-pair mask), and a second kernel, one warp per atom,
//     evaluates the listed pairs in FP64 from the stored coordinates, exactly as the oracle
//     sees them, so the filter only has to be conservative and never holds a warp on an
//     FP64 dependency chain; an atom with more hits than its list holds is rescanned against
//     all j by its warp, so nothing is ever dropped;
//   * each thread carries R atoms i in registers (one shared-memory load feeds 3R FFMA);
//   * the j chunks are dealt round-robin to blockIdx.y so that 148 SMs are busy and the dense
//     (nearby) chunks are spread evenly.
// k_force_allpairs_general is the unsorted per-pair-minimum-image variant for boxes too small
// to pre-shift (L/2 - rc smaller than a block) and the cross-check of the tiled kernel.
#include <math.h>
#include "common.cuh"
#include "pair.cuh"

#define AP_T 128      // threads per block of the general kernel
#ifndef AP_FT
#define AP_FT 32      // threads per block of the sorted filter kernel: one warp (a block retires with its warp)
#endif
#define AP_TJ 32      // j atoms per staged chunk: one per lane
#define AP_BPS (5 * 128 / AP_FT)   // resident filter blocks per SM (register bound, R = 8: 20 warps)
#define AP_ET 256     // threads per block of the list evaluation kernel (32 atoms)
#define FULLMASK 0xffffffffu

// ---------------------------------------------------------------------------------------
// General variant: per-pair minimum image, valid for any rc <= L/2 and any atom order.
__global__ void __launch_bounds__(AP_T)
k_force_allpairs_general(const float4 *__restrict__ pos, int N, PairParams P, float L, float invL,
                         double Ld, double invLd, int jchunk, double *__restrict__ fpart,
                         double *__restrict__ part_pe, double *__restrict__ part_w, unsigned *__restrict__ tile_done,
                         float4 *__restrict__ frc)
{
    __shared__ float4 tile[AP_T];
    __shared__ double red[32];
    __shared__ int last_of_tile;
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
        // 32 j at a time: an FP32 pass marks the candidates in a bit mask, then every lane walks its own bits.  With
        // the FP64 evaluation inside the distance loop a warp took that (long, divergent) branch on nearly every j,
        // because some lane or other had a hit; now it takes it max-over-lanes(hits) times: ~8 instead of ~31 per 32 j
        // at liquid density.  Each lane still adds its pairs in ascending j: the sums are unchanged to the bit.
        for (int k0 = 0; k0 < cnt; k0 += 32) {
            const int kn = min(32, cnt - k0);
            unsigned hits = 0u;
#pragma unroll 8
            for (int k = 0; k < kn; k++) {
                const float4 pj = tile[k0 + k];
                float dx = pj.x - pi.x, dy = pj.y - pi.y, dz = pj.z - pi.z;
                dx = fmaf(-L, rintf(dx * invL), dx);
                dy = fmaf(-L, rintf(dy * invL), dy);
                dz = fmaf(-L, rintf(dz * invL), dz);
                const float r2 = fmaf(dx, dx, fmaf(dy, dy, dz * dz));
                hits |= (r2 < P.rc2f_filter && (j0 + k0 + k) != i) ? (1u << k) : 0u;
            }
            while (hits) {
                const int k = __ffs(hits) - 1;
                hits &= hits - 1u;
                const float4 pj = tile[k0 + k];
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
    // Combination of the j splits inside this launch (it was a kernel of its own: one launch less per step, which
    // is what a small system's step consists of): the block that arrives last on this tile of atoms sums
    // the tile's partial forces in split order -- the same sum whoever that is -- and puts the counter back to zero
    // for the next launch.
    __threadfence();
    __syncthreads();
    if (tid == 0) last_of_tile = atomicAdd(&tile_done[blockIdx.x], 1u) == gridDim.y - 1;
    __syncthreads();
    if (!last_of_tile) return;
    __threadfence();
    if (live) {
        double sx = 0.0, sy = 0.0, sz = 0.0;
        for (int s = 0; s < (int)gridDim.y; s++) {
            const size_t base = (size_t)s * 3 * N;
            sx += __ldcg(&fpart[base + i]);
            sy += __ldcg(&fpart[base + (size_t)N + i]);
            sz += __ldcg(&fpart[base + 2 * (size_t)N + i]);
        }
        frc[i] = make_float4((float)sx, (float)sy, (float)sz, 0.0f);
    }
    if (tid == 0) tile_done[blockIdx.x] = 0u;
}

// ---------------------------------------------------------------------------------------
// Spatial sort: counting sort of the state by the Hilbert index of a cell on a 2^b grid
// (side L / 2^b in [1.5, 3) sigma), so that any run of consecutive atoms is spatially compact
// (a Hilbert curve has no jumps, unlike Morton order).
struct SortGrid { int bits; float scale; };   // 2^bits cells per dimension, scale = 2^bits / L

// Hilbert index of cell (x, y, z) on a 2^b cube: Skilling's axes-to-transpose transform
// (AIP Conf. Proc. 707, 381 (2004)) followed by bit interleaving.
__device__ __forceinline__ unsigned hilbert3(unsigned x, unsigned y, unsigned z, int b)
{
    unsigned X[3] = {x, y, z};
    const unsigned M = 1u << (b - 1);
    for (unsigned Q = M; Q > 1; Q >>= 1) {
        const unsigned P = Q - 1;
#pragma unroll
        for (int i = 0; i < 3; i++) {
            if (X[i] & Q) X[0] ^= P;
            else { unsigned t = (X[0] ^ X[i]) & P; X[0] ^= t; X[i] ^= t; }
        }
    }
    X[1] ^= X[0];
    X[2] ^= X[1];
    unsigned t = 0;
    for (unsigned Q = M; Q > 1; Q >>= 1)
        if (X[2] & Q) t ^= Q - 1;
    X[0] ^= t; X[1] ^= t; X[2] ^= t;
    unsigned h = 0;
    for (int k = b - 1; k >= 0; k--)
        h = (h << 3) | (((X[0] >> k) & 1u) << 2) | (((X[1] >> k) & 1u) << 1) | ((X[2] >> k) & 1u);
    return h;
}

__global__ void __launch_bounds__(256)
k_bin_hilbert(const float4 *__restrict__ pos, int N, SortGrid g, int *__restrict__ bin_of, int *__restrict__ rank,
              int *__restrict__ count)
{
    int i = blockIdx.x * 256 + threadIdx.x;
    if (i >= N) return;
    float4 p = pos[i];
    const int n = 1 << g.bits;
    unsigned cx = min(n - 1, (int)(p.x * g.scale));
    unsigned cy = min(n - 1, (int)(p.y * g.scale));
    unsigned cz = min(n - 1, (int)(p.z * g.scale));
    int b = (g.bits > 0) ? (int)hilbert3(cx, cy, cz, g.bits) : 0;
    bin_of[i] = b;
    rank[i] = atomicAdd(&count[b], 1);
}

__global__ void __launch_bounds__(256)
k_scatter_sorted(const float4 *__restrict__ pos, const float4 *__restrict__ vel, int N, const int *__restrict__ bin_of,
                 const int *__restrict__ rank, const int *__restrict__ start, float4 *__restrict__ pos2,
                 float4 *__restrict__ vel2)
{
    int i = blockIdx.x * 256 + threadIdx.x;
    if (i >= N) return;
    int dst = start[bin_of[i]] + rank[i];
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

template <int R>
__global__ void __launch_bounds__(AP_FT, AP_BPS)
k_allpairs_filter(const float4 *__restrict__ pos, int N, float rc, float rc2, float L, float invL, float hmax,
                  int nchunks_j, int *__restrict__ nbr_count, int *__restrict__ nbr_list, int cap)
{
    __shared__ float4 tile[(AP_FT / 32) * 2 * AP_TJ];                    // [4 warps][2][AP_TJ]
    __shared__ float bb[(AP_FT / 32) * 6];

    const int tid = threadIdx.x, lane = tid & 31, wid = tid >> 5;
    const int split = blockIdx.y, nsplit = gridDim.y;
    const int bbase = blockIdx.x * (AP_FT * R);
    const int i0 = bbase + wid * (32 * R) + lane;                        // atom r of this lane: i0 + 32 r

    // ---- block geometry: periodic bounding box of the block's atoms.  Per dimension, a
    // 32-bin occupancy mask locates the longest empty stretch of the circle [0,L); cutting the
    // circle in its middle unwraps the coordinates, whatever images the atoms are stored as.
    float ux[R], uy[R], uz[R];
    unsigned occ[3] = {0u, 0u, 0u};
    const float binscale = 32.f * invL;
#pragma unroll
    for (int r = 0; r < R; r++) {
        const int i = i0 + 32 * r;
        ux[r] = uy[r] = uz[r] = 0.f;
        if (i < N) {
            const float4 p = pos[i];
            ux[r] = p.x; uy[r] = p.y; uz[r] = p.z;
            occ[0] |= 1u << min(31, (int)(p.x * binscale));
            occ[1] |= 1u << min(31, (int)(p.y * binscale));
            occ[2] |= 1u << min(31, (int)(p.z * binscale));
        }
    }
#pragma unroll
    for (int d = 0; d < 3; d++) occ[d] = __reduce_or_sync(FULLMASK, occ[d]);
    unsigned *bbu = (unsigned *)bb;
    if (lane == 0) {
#pragma unroll
        for (int d = 0; d < 3; d++) bbu[wid * 3 + d] = occ[d];
    }
    __syncthreads();
    float cut[3];
    bool compact = true;
#pragma unroll
    for (int d = 0; d < 3; d++) {
        unsigned m = 0u;
#pragma unroll
        for (int k = 0; k < AP_FT / 32; k++) m |= bbu[k * 3 + d];
        unsigned e = ~m, last = e;
        int len = 0;
        while (e) {                                  // bit i of e: bins i .. i+len all empty (cyclic)
            last = e;
            e &= (e >> 1) | (e << 31);
            len++;
        }
        if (len == 0) { compact = false; cut[d] = 0.f; }
        else cut[d] = ((float)(__ffs(last) - 1) + 0.5f * (float)len) * (L * 0.03125f);
    }
    __syncthreads();
    float mn[3] = {INFINITY, INFINITY, INFINITY}, mx[3] = {-INFINITY, -INFINITY, -INFINITY};
#pragma unroll
    for (int r = 0; r < R; r++) {
        if (i0 + 32 * r < N) {
            float x = ux[r] - cut[0], y = uy[r] - cut[1], z = uz[r] - cut[2];
            x += (x < 0.f) ? L : 0.f; y += (y < 0.f) ? L : 0.f; z += (z < 0.f) ? L : 0.f;
            mn[0] = fminf(mn[0], x); mx[0] = fmaxf(mx[0], x);
            mn[1] = fminf(mn[1], y); mx[1] = fmaxf(mx[1], y);
            mn[2] = fminf(mn[2], z); mx[2] = fmaxf(mx[2], z);
        }
    }
#pragma unroll
    for (int d = 0; d < 3; d++) {
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) {
            mn[d] = fminf(mn[d], __shfl_xor_sync(FULLMASK, mn[d], o));
            mx[d] = fmaxf(mx[d], __shfl_xor_sync(FULLMASK, mx[d], o));
        }
    }
    if (lane == 0) {
#pragma unroll
        for (int d = 0; d < 3; d++) { bb[wid * 6 + d] = mn[d]; bb[wid * 6 + 3 + d] = mx[d]; }
    }
    __syncthreads();
    float cen[3], hm = 0.f;
#pragma unroll
    for (int d = 0; d < 3; d++) {
        mn[d] = bb[d]; mx[d] = bb[3 + d];
#pragma unroll
        for (int k = 1; k < AP_FT / 32; k++) {
            mn[d] = fminf(mn[d], bb[k * 6 + d]);
            mx[d] = fmaxf(mx[d], bb[k * 6 + 3 + d]);
        }
        cen[d] = cut[d] + 0.5f * (mn[d] + mx[d]);
        hm = fmaxf(hm, 0.5f * (mx[d] - mn[d]));
    }
    // the image of j nearest the centre is the minimum image for every i of the block when
    // half extent + rc <= L/2 (with slack); otherwise this block tests per-pair minimum images
    const bool preshift = compact && hm <= hmax;
    const float cx = cen[0], cy = cen[1], cz = cen[2];                  // block centre (any image)

    // filter threshold: rc^2 plus the rounding error of the 3-FFMA form at these magnitudes
    const float rcf = rc;
    const float Mi = 1.7320508f * hm, M = Mi + rcf;
    const float thr = rc2 + 2e-6f * (M * M + 2.f * M * Mi) + 8.f * rcf * (L * 1.1920929e-7f) + 1e-6f * rc2;

    float ax[R], ay[R], az[R], T[R];
#pragma unroll
    for (int r = 0; r < R; r++) {
        float x = ux[r] - cx, y = uy[r] - cy, z = uz[r] - cz;
        x = fmaf(-L, rintf(x * invL), x);
        y = fmaf(-L, rintf(y * invL), y);
        z = fmaf(-L, rintf(z * invL), z);
        ax[r] = -2.f * x; ay[r] = -2.f * y; az[r] = -2.f * z;
        T[r] = (i0 + 32 * r < N) ? thr - fmaf(x, x, fmaf(y, y, z * z)) : -INFINITY;
    }

    // stage one chunk of 32 j atoms (per warp): u = image of x_j nearest the centre,
    // w = |u|^2 (padding: w = +inf).  The global load of the next chunk is issued before the
    // current one is processed, the shared-memory store after it.
    auto chunk_load = [&](int jc) {
        const int j = min(jc * AP_TJ + lane, N - 1);
        return pos[j];
    };
    auto chunk_store = [&](float4 *dst, const float4 p, bool valid) {
        float4 u;
        u.x = p.x - cx; u.y = p.y - cy; u.z = p.z - cz;
        u.x = fmaf(-L, rintf(u.x * invL), u.x);
        u.y = fmaf(-L, rintf(u.y * invL), u.y);
        u.z = fmaf(-L, rintf(u.z * invL), u.z);
        u.w = valid ? fmaf(u.x, u.x, fmaf(u.y, u.y, u.z * u.z)) : INFINITY;
        dst[lane] = u;
    };

    // append the hits of one chunk to the lists of this lane's atoms: one atomic per non-empty
    // mask reserves the slots (all R issued before any result is used), then the j indices
    // are stored; slots beyond the capacity are counted but not stored (k_allpairs_eval then
    // rescans that atom)
    auto append = [&](unsigned (&mk)[R], int jbase) {
        int base[R];
#pragma unroll
        for (int r = 0; r < R; r++) {
            const int i = i0 + 32 * r;
            const int self = i - jbase;                                 // the pair (i, i) is not a pair
            if (self >= 0 && self < 32) mk[r] &= ~(1u << self);
            base[r] = 0;
            if (mk[r]) base[r] = atomicAdd(nbr_count + i, __popc(mk[r]));
        }
#pragma unroll
        for (int r = 0; r < R; r++) {
            unsigned m2 = mk[r];
            int *row = nbr_list + (size_t)(i0 + 32 * r) * cap;
            int b = base[r];
            while (m2) {
                const int k = __ffs(m2) - 1;
                m2 &= m2 - 1u;
                if (b < cap) row[b] = jbase + k;
                b++;
            }
        }
    };

    int buf = 0;
    float4 *wtile = tile + wid * (2 * AP_TJ);
    if (split < nchunks_j) chunk_store(wtile, chunk_load(split), split * AP_TJ + lane < N);
    __syncwarp();
    for (int jc = split; jc < nchunks_j; jc += nsplit) {
        const float4 *tc = wtile + buf * AP_TJ;
        const int jn = jc + nsplit;
        const bool have_next = jn < nchunks_j;
        float4 pnext = make_float4(0.f, 0.f, 0.f, 0.f);
        if (have_next) pnext = chunk_load(jn);
        do {
            if (preshift) {
                float m[R];
#pragma unroll
                for (int r = 0; r < R; r++) m[r] = INFINITY;
#pragma unroll 4
                for (int k = 0; k < 32; k += 2) {
                    const float4 a = tc[k], b = tc[k + 1];
                    if constexpr (R >= 2) {
                        // two atoms per FFMA2 (same IEEE fma per half as the scalar rescan below)
                        const float2 aX = make_float2(a.x, a.x), aY = make_float2(a.y, a.y), aZ = make_float2(a.z, a.z),
                                     aW = make_float2(a.w, a.w);
                        const float2 bX = make_float2(b.x, b.x), bY = make_float2(b.y, b.y), bZ = make_float2(b.z, b.z),
                                     bW = make_float2(b.w, b.w);
#pragma unroll
                        for (int q = 0; q < R / 2; q++) {
                            const float2 x2 = make_float2(ax[2 * q], ax[2 * q + 1]), y2 = make_float2(ay[2 * q], ay[2 * q + 1]),
                                         z2 = make_float2(az[2 * q], az[2 * q + 1]);
                            const float2 v1 = __ffma2_rn(x2, aX, __ffma2_rn(y2, aY, __ffma2_rn(z2, aZ, aW)));
                            const float2 v2 = __ffma2_rn(x2, bX, __ffma2_rn(y2, bY, __ffma2_rn(z2, bZ, bW)));
                            m[2 * q] = fminf(m[2 * q], fminf(v1.x, v2.x));
                            m[2 * q + 1] = fminf(m[2 * q + 1], fminf(v1.y, v2.y));
                        }
                    } else {
#pragma unroll
                        for (int r = 0; r < R; r++) {
                            float v1 = fmaf(ax[r], a.x, fmaf(ay[r], a.y, fmaf(az[r], a.z, a.w)));
                            float v2 = fmaf(ax[r], b.x, fmaf(ay[r], b.y, fmaf(az[r], b.z, b.w)));
                            m[r] = fminf(m[r], fminf(v1, v2));
                        }
                    }
                }
                bool hit = false;
#pragma unroll
                for (int r = 0; r < R; r++) hit |= m[r] < T[r];
                if (!__any_sync(FULLMASK, hit)) break;
                // some pair of this chunk is inside the threshold: rescan into hit masks
                const int jbase = jc * AP_TJ;
                unsigned mk[R];
#pragma unroll
                for (int r = 0; r < R; r++) {
                    mk[r] = 0u;
                    if (__any_sync(FULLMASK, m[r] < T[r])) {
#pragma unroll 4
                        for (int k = 0; k < 32; k++) {
                            const float4 a = tc[k];
                            float v = fmaf(ax[r], a.x, fmaf(ay[r], a.y, fmaf(az[r], a.z, a.w)));
                            mk[r] |= (v < T[r]) ? (1u << k) : 0u;
                        }
                    }
                }
                append(mk, jbase);
            } else {
                // block not compact (too wide for this box): per-pair minimum image on the
                // centred coordinates
                const int jbase = jc * AP_TJ;
                unsigned mk[R];
#pragma unroll
                for (int r = 0; r < R; r++) {
                    mk[r] = 0u;
                    if (T[r] == -INFINITY) continue;
                    for (int k = 0; k < 32; k++) {
                        const float4 a = tc[k];
                        float dx = fmaf(0.5f, ax[r], a.x), dy = fmaf(0.5f, ay[r], a.y), dz = fmaf(0.5f, az[r], a.z);
                        dx = fmaf(-L, rintf(dx * invL), dx);
                        dy = fmaf(-L, rintf(dy * invL), dy);
                        dz = fmaf(-L, rintf(dz * invL), dz);
                        float r2 = fmaf(dx, dx, fmaf(dy, dy, dz * dz));
                        mk[r] |= (r2 < thr && a.w != INFINITY) ? (1u << k) : 0u;
                    }
                }
                append(mk, jbase);
            }
        } while (false);
        if (have_next) chunk_store(wtile + (buf ^ 1) * AP_TJ, pnext, jn * AP_TJ + lane < N);
        __syncwarp();
        buf ^= 1;
    }
}

// Eight lanes per atom: evaluate the listed candidate pairs in FP64 (Eq. 1-3)
// from the stored coordinates, two independent chains per lane, reduce over the eight lanes,
// write the force, reset the counter.
#define AP_EL 8       // lanes per atom
__global__ void __launch_bounds__(AP_ET)
k_allpairs_eval(const float4 *__restrict__ pos, int N, PairParams P, double Ld, double invLd,
                int *__restrict__ nbr_count, const int *__restrict__ nbr_list, int cap, float4 *__restrict__ frc,
                double *__restrict__ part_pe, double *__restrict__ part_w)
{
    __shared__ double red[32];
    const int sub = threadIdx.x & (AP_EL - 1);
    const int i = blockIdx.x * (AP_ET / AP_EL) + (threadIdx.x / AP_EL);
    double fx = 0.0, fy = 0.0, fz = 0.0, pe = 0.0, w = 0.0;
    double gx = 0.0, gy = 0.0, gz = 0.0, pe2 = 0.0, w2 = 0.0;
    if (i < N) {
        const int n = nbr_count[i];
        const float4 pi = pos[i];
        if (n <= cap) {
            const int *row = nbr_list + (size_t)i * cap;
            int k = sub;
            for (; k + AP_EL < n; k += 2 * AP_EL) {
                const int ja = row[k], jb = row[k + AP_EL];
                const float4 pa = pos[ja], pb = pos[jb];
                ap_exact(P, pi, pa, Ld, invLd, fx, fy, fz, pe, w);
                ap_exact(P, pi, pb, Ld, invLd, gx, gy, gz, pe2, w2);
            }
            if (k < n) ap_exact(P, pi, pos[row[k]], Ld, invLd, fx, fy, fz, pe, w);
        } else {
            // more candidates than the list holds: test every j (slow, never wrong)
            for (int j = sub; j < N; j += AP_EL)
                if (j != i) ap_exact(P, pi, pos[j], Ld, invLd, fx, fy, fz, pe, w);
        }
    }
    fx += gx; fy += gy; fz += gz; pe += pe2; w += w2;
#pragma unroll
    for (int o = AP_EL / 2; o > 0; o >>= 1) {
        fx += __shfl_xor_sync(FULLMASK, fx, o);
        fy += __shfl_xor_sync(FULLMASK, fy, o);
        fz += __shfl_xor_sync(FULLMASK, fz, o);
    }
    if (i < N && sub == 0) {
        frc[i] = make_float4((float)fx, (float)fy, (float)fz, 0.0f);
        nbr_count[i] = 0;                           // ready for the next force evaluation
    }
    pe = block_sum(pe, red);
    w = block_sum(w, red);
    if (threadIdx.x == 0) {
        part_pe[blockIdx.x] = 0.5 * pe;             // every pair is visited from both ends
        part_w[blockIdx.x] = 0.5 * w;
    }
}

// ---------------------------------------------------------------------------------------
// Host side: choose R and the j split (md_create), sort, launch.
static int ap_sm_count()
{
    static int sms = 0;
    if (!sms) {
        int dev = 0;
        if (cudaGetDevice(&dev) != cudaSuccess || cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess ||
            sms <= 0)
            sms = 148;
    }
    return sms;
}

// i blocks and j splits for R atoms per thread: one wave of AP_BPS resident blocks per SM
static void ap_shape(int64_t N, int R, int *iblocks, int *tsplit)
{
    const int ib = (int)((N + AP_FT * R - 1) / (AP_FT * R));
    const int ntj = (int)((N + AP_TJ - 1) / AP_TJ);
    int k = (AP_BPS * ap_sm_count()) / ib;
    if (k > ntj / 4) k = ntj / 4;                                   // at least 4 chunks per warp
    if (k > 64) k = 64;
    if (k < 1) k = 1;
    *iblocks = ib;
    *tsplit = k;
}

void ljmd_ap_set_R(md_sim *s, int R)
{
    s->ap_R = R;
    s->ap_tiled = R > 0;
    s->ap_ntiles = 0;
    s->ap_tsplit = 1;
    if (R > 0) ap_shape(s->N, R, &s->ap_ntiles, &s->ap_tsplit);
}

void ljmd_ap_plan(md_sim *s)
{
    const double L = s->L, rc = s->rc;
    const double slack = 0.05 * rc;
    s->ap_hmax = (float)(0.5 * L - rc - slack);
    ljmd_ap_set_R(s, 0);
    s->ap_sort_g = 0;
    s->ap_sort_bins = 1;
    if (s->N >= (1LL << 30)) return;
    // Hilbert grid: 2^b cells per dimension with side L / 2^b in [1.5, 3) sigma, b <= 6
    int bits = 0;
    while (bits < 6 && L / (double)(1 << (bits + 1)) >= 1.5) bits++;
    s->ap_sort_g = bits;
    s->ap_sort_bins = 1 << (3 * bits);
    // largest R whose block of 128 R consecutive atoms (a cube of that volume, stretched by
    // the Hilbert curve and the cell granularity) still fits the pre-shift bound; a block that
    // turns out not to fit falls back to per-pair minimum images inside the kernel
    const double vol_per_atom = L * L * L / (double)s->N;
    for (int R = 8; R >= 1; R >>= 1) {
        double side = cbrt((double)AP_FT * R * vol_per_atom);
        double h = 0.5 * side * 1.2 + 0.5 * L / (double)(1 << bits) + 0.3;   // 0.3: drift between re-sorts
        if (h <= s->ap_hmax && s->N >= AP_FT * R) { ljmd_ap_set_R(s, R); break; }
    }
}

static int ap_sort(md_sim *s)
{
    int N = (int)s->N;
    int nb = (N + 255) / 256;
    SortGrid g;
    g.bits = s->ap_sort_g;
    g.scale = (float)((double)(1 << g.bits) / s->L);
    k_bin_hilbert<<<nb, 256, 0, s->stream>>>(s->pos, N, g, s->cell_of, s->rank, s->tile_count);
    CKL(s);
    int r = ljmd_scan_counts(s, s->tile_count, s->tile_start, s->ap_sort_bins);
    if (r) return r;
    k_scatter_sorted<<<nb, 256, 0, s->stream>>>(s->pos, s->vel, N, s->cell_of, s->rank, s->tile_start, s->pos2, s->vel2);
    CKL(s);
    float4 *t = s->pos; s->pos = s->pos2; s->pos2 = t;
    t = s->vel; s->vel = s->vel2; s->vel2 = t;
    return MD_OK;
}

template <int R>
static int ap_launch(md_sim *s)
{
    const int N = (int)s->N;
    dim3 grid(s->ap_ntiles, s->ap_tsplit);
    k_allpairs_filter<R><<<grid, AP_FT, 0, s->stream>>>(s->pos, N, (float)s->rc, (float)(s->rc * s->rc), s->Lf, 1.0f / s->Lf,
                                                      s->ap_hmax, (N + AP_TJ - 1) / AP_TJ, s->nbr_count, s->nbr_list,
                                                      s->nbr_cap);
    CKL(s);
    return MD_OK;
}

// Candidate lists of the sorted kernel, allocated on first use: per atom, room for 2.5 times
// the mean number of atoms inside rc (at least 64), a multiple of 32.
static int ap_alloc_lists(md_sim *s)
{
    if (s->nbr_list) return MD_OK;
    const double mean = 4.0 / 3.0 * 3.14159265358979 * s->rc * s->rc * s->rc * (double)s->N / (s->L * s->L * s->L);
    int cap = (int)(2.5 * mean) + 32;
    if (cap < 64) cap = 64;
    cap = (cap + 31) / 32 * 32;
    s->nbr_cap = cap;
    s->nbr_count = (int *)ljmd_dev_alloc((size_t)s->N * sizeof(int), s->stream);
    s->nbr_list = (int *)ljmd_dev_alloc((size_t)s->N * cap * sizeof(int), s->stream);
    if (!s->nbr_count || !s->nbr_list) {
        ljmd_dev_free(s->nbr_count, s->stream);
        ljmd_dev_free(s->nbr_list, s->stream);
        s->nbr_count = s->nbr_list = nullptr;
        return MD_ENOMEM;
    }
    CK(cudaMemsetAsync(s->nbr_count, 0, (size_t)s->N * sizeof(int), s->stream));
    return MD_OK;
}

int ljmd_forces_allpairs(md_sim *s)
{
    int N = (int)s->N;
    double *ppe = s->part + (size_t)s->part_cap;
    double *pw = s->part + 2 * (size_t)s->part_cap;
    if (s->ap_tiled && !s->ap_force_general) {
        int r = ap_alloc_lists(s);
        if (r) return r;
        if (s->layout != LAYOUT_TILE || s->ap_since_sort >= s->sort_every) {
            if ((r = ap_sort(s))) return r;
            s->layout = LAYOUT_TILE;
            s->ap_since_sort = 0;
            ljmd_tick(s, TAG_BUILD);
        }
        s->ap_since_sort++;
        switch (s->ap_R) {
        case 8: r = ap_launch<8>(s); break;
        case 4: r = ap_launch<4>(s); break;
        case 2: r = ap_launch<2>(s); break;
        default: r = ap_launch<1>(s); break;
        }
        if (r) return r;
        ljmd_tick(s, TAG_FORCE);
        const int nb = (N + AP_ET / AP_EL - 1) / (AP_ET / AP_EL);
        k_allpairs_eval<<<nb, AP_ET, 0, s->stream>>>(s->pos, N, s->pp, s->L, 1.0 / s->L, s->nbr_count, s->nbr_list,
                                                    s->nbr_cap, s->frc, ppe, pw);
        CKL(s);
        s->n_pe = nb;
        ljmd_tick(s, TAG_FORCE2);
    } else {
        int niblk = (N + AP_T - 1) / AP_T;
        int nsplit = s->ap_nsplit;
        int jchunk = (N + nsplit - 1) / nsplit;
        jchunk = (jchunk + 31) / 32 * 32;
        dim3 grid(niblk, nsplit);
        k_force_allpairs_general<<<grid, AP_T, 0, s->stream>>>(s->pos, N, s->pp, s->Lf, 1.0f / s->Lf, s->L, 1.0 / s->L,
                                                              jchunk, s->fpart, ppe, pw, s->ap_tile_done, s->frc);
        CKL(s);
        s->n_pe = niblk * nsplit;
        if (s->layout == LAYOUT_CELL || s->layout == LAYOUT_VERLET) s->layout = LAYOUT_NONE;   // lpos no longer tracked
        ljmd_tick(s, TAG_FORCE);
    }
    return MD_OK;
}
