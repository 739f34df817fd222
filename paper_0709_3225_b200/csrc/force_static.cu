// md_forces_allpairs_static: the all-pairs Lennard-Jones evaluation (PAPER.md:49-52,
// Eq. 1, and :56-61, Eq. 2-3) for callers that must not allocate device memory.
//
// Who that is.  Some programs hand the whole card to a memory pool of their own when they start (a serving
// process, a framework with a pre-reserved arena), so a cudaMalloc from a library they call fails for lack of
// memory; others run inside a loop with a latency budget, where cudaMalloc and cudaFree are forbidden because
// both stall the whole device while they run.  md_create and every md_* call on a handle allocate; this entry
// point does not: no cudaMalloc, cudaFree, or allocating library routine, on any call.
//
// How.  It is a variant of k_force_allpairs_general (force_allpairs.cu): the same j-split with per-pair
// minimum images and every in-range pair evaluated in FP64, but the scratch that kernel takes from md_create
// (partial forces of the j splits, block partials of PE and W) lives in ONE file-scope __device__ array of
// fixed size, g_static_scratch below.  The array is part of the library image: every GPU on which the
// library's code is loaded holds its SA_SCRATCH_DOUBLES * 8 = 1,319,936 bytes until the process exits.
// The fixed size is where the limit N <= MD_STATIC_MAX_ATOMS comes from.
//
// The combination of the j splits is folded into the same launch: the block that arrives last on a tile of
// 128 atoms i (a counter per tile, in the scratch) sums that tile's partial forces in split order, and the
// block that arrives last of all sums the energy partials in block order, so the result does not depend on
// which block that was.  One memset (of the counters) and one kernel per call.
//
// Sharing.  All calls on a device use the same array and it keeps what the last call left in it.  The only
// part that has to start at zero, the arrival counters, is cleared at the start of every call, on the call's
// stream; everything else is written before it is read.  Two calls that overlap on the GPU (from two host
// threads, on two streams) race on the array and both results are then undefined: serialise them.
#include <math.h>
#include <string.h>
#include <mutex>
#include "common.cuh"
#include "pair.cuh"

#define SA_T 128                     // threads per block = atoms i per tile = largest j chunk staged at once
#define SA_MAX_TILES (MD_STATIC_MAX_ATOMS / SA_T)
#define SA_TARGET_BLOCKS 296         // two blocks per SM of a B200
#define SA_MAX_BLOCKS 512            // >= SA_TARGET_BLOCKS + SA_MAX_TILES
// layout of the scratch, in doubles
#define SA_OFF_CTR 0                 // 256 unsigned: tile_done[SA_MAX_TILES], then all_done
#define SA_CTR_DOUBLES 128
#define SA_OFF_PE (SA_OFF_CTR + SA_CTR_DOUBLES)
#define SA_OFF_W (SA_OFF_PE + SA_MAX_BLOCKS)
#define SA_OFF_FPART (SA_OFF_W + SA_MAX_BLOCKS)
// nsplit <= SA_TARGET_BLOCKS / tiles + 1, so nsplit * 3 * N <= 3 * (SA_TARGET_BLOCKS * SA_T + N)
#define SA_FPART_DOUBLES (3 * (SA_TARGET_BLOCKS * SA_T + MD_STATIC_MAX_ATOMS))
#define SA_SCRATCH_DOUBLES (SA_OFF_FPART + SA_FPART_DOUBLES)

static_assert(SA_MAX_TILES + 1 <= 2 * SA_CTR_DOUBLES, "counters do not fit their region");
static_assert(SA_TARGET_BLOCKS + SA_MAX_TILES <= SA_MAX_BLOCKS, "energy partials do not fit their region");

// The scratch.  In host code this name is only a stand-in for the symbol, NOT a device address: the address a
// kernel can use comes from cudaGetSymbolAddress (static_scratch_ptr below).
static __device__ __align__(256) double g_static_scratch[SA_SCRATCH_DOUBLES];

// pos, frc: [N][3] floats in device memory; pe_w: 2 doubles in device memory.  grid = (tiles, nsplit).
__global__ void __launch_bounds__(SA_T)
k_force_allpairs_static(const float *__restrict__ pos, int N, PairParams P, float L, float invL, double Ld, double invLd,
                        int jchunk, double *__restrict__ scratch, float *__restrict__ frc, double *__restrict__ pe_w)
{
    __shared__ float tx[SA_T], ty[SA_T], tz[SA_T];
    __shared__ double red[32];
    __shared__ int last_of_tile, last_of_all;
    unsigned *tile_done = (unsigned *)(scratch + SA_OFF_CTR);
    unsigned *all_done = tile_done + SA_MAX_TILES;
    double *part_pe = scratch + SA_OFF_PE, *part_w = scratch + SA_OFF_W, *fpart = scratch + SA_OFF_FPART;

    const int tid = threadIdx.x;
    const int i = blockIdx.x * SA_T + tid;
    const int jbeg = blockIdx.y * jchunk;
    const int jend = min(N, jbeg + jchunk);
    const bool live = i < N;
    float xi = 0.f, yi = 0.f, zi = 0.f;
    if (live) { xi = pos[3 * i]; yi = pos[3 * i + 1]; zi = pos[3 * i + 2]; }
    double fx = 0.0, fy = 0.0, fz = 0.0, pe = 0.0, w = 0.0;

    for (int j0 = jbeg; j0 < jend; j0 += SA_T) {
        const int cnt = min(SA_T, jend - j0);
        __syncthreads();
        if (tid < cnt) {
            tx[tid] = pos[3 * (j0 + tid)];
            ty[tid] = pos[3 * (j0 + tid) + 1];
            tz[tid] = pos[3 * (j0 + tid) + 2];
        }
        __syncthreads();
        if (!live) continue;
        // 32 j at a time: an FP32 pass marks the candidates in a bit mask, then every lane walks its own bits (the warp
        // takes the long FP64 branch max-over-lanes(hits) times instead of on nearly every j)
        for (int k0 = 0; k0 < cnt; k0 += 32) {
            const int kn = min(32, cnt - k0);
            unsigned hits = 0u;
#pragma unroll 8
            for (int k = 0; k < kn; k++) {
                float dx = tx[k0 + k] - xi, dy = ty[k0 + k] - yi, dz = tz[k0 + k] - zi;
                dx = fmaf(-L, rintf(dx * invL), dx);
                dy = fmaf(-L, rintf(dy * invL), dy);
                dz = fmaf(-L, rintf(dz * invL), dz);
                const float r2 = fmaf(dx, dx, fmaf(dy, dy, dz * dz));
                hits |= (r2 < P.rc2f_filter && (j0 + k0 + k) != i) ? (1u << k) : 0u;
            }
            while (hits) {
                const int k = k0 + __ffs(hits) - 1;
                hits &= hits - 1u;
                // the FP32 test only has to be conservative: the pair is decided and evaluated in FP64
                // from the coordinates as stored
                double ex = (double)tx[k] - (double)xi, ey = (double)ty[k] - (double)yi, ez = (double)tz[k] - (double)zi;
                ex = fma(-Ld, rint(ex * invLd), ex);
                ey = fma(-Ld, rint(ey * invLd), ey);
                ez = fma(-Ld, rint(ez * invLd), ez);
                pair_f64(P, ex, ey, ez, fx, fy, fz, pe, w);
            }
        }
    }
    if (live) {
        const size_t base = (size_t)blockIdx.y * 3 * N;
        fpart[base + i] = fx;
        fpart[base + (size_t)N + i] = fy;
        fpart[base + 2 * (size_t)N + i] = fz;
    }
    pe = block_sum(pe, red);
    w = block_sum(w, red);
    const int nblocks = gridDim.x * gridDim.y;
    if (tid == 0) {
        const int b = blockIdx.y * gridDim.x + blockIdx.x;
        part_pe[b] = 0.5 * pe;                 // every pair is visited from both ends
        part_w[b] = 0.5 * w;
    }
    // arrival: this block's partials are visible device-wide before its tickets are drawn
    __threadfence();
    __syncthreads();
    if (tid == 0) {
        last_of_tile = atomicAdd(&tile_done[blockIdx.x], 1u) == gridDim.y - 1;
        last_of_all = atomicAdd(all_done, 1u) == (unsigned)nblocks - 1;
    }
    __syncthreads();
    if (last_of_tile) {
        __threadfence();
        if (live) {
            double sx = 0.0, sy = 0.0, sz = 0.0;
            for (int s = 0; s < (int)gridDim.y; s++) {          // split order: the same sum whoever came last
                const size_t base = (size_t)s * 3 * N;
                sx += __ldcg(&fpart[base + i]);
                sy += __ldcg(&fpart[base + (size_t)N + i]);
                sz += __ldcg(&fpart[base + 2 * (size_t)N + i]);
            }
            frc[3 * i] = (float)sx;
            frc[3 * i + 1] = (float)sy;
            frc[3 * i + 2] = (float)sz;
        }
    }
    if (last_of_all) {
        __threadfence();
        double a = 0.0, c = 0.0;
        for (int b = tid; b < nblocks; b += SA_T) {
            a += __ldcg(&part_pe[b]);
            c += __ldcg(&part_w[b]);
        }
        a = block_sum(a, red);
        c = block_sum(c, red);
        if (tid == 0) {
            pe_w[0] = a;
            pe_w[1] = c;
        }
    }
}

// Device address of g_static_scratch on the current device.  Looked up once per device, with that device
// current, and checked: the symbol's name itself is not an address host code may pass to a kernel.
static int static_scratch_ptr(double **out)
{
    static std::mutex mu;
    static double *ptr[64] = {nullptr};
    int dev = 0;
    CK(cudaGetDevice(&dev));
    if (dev < 0 || dev >= 64) return MD_EUNSUPPORTED;
    std::lock_guard<std::mutex> lock(mu);
    if (!ptr[dev]) {
        double *p = nullptr;
        CK(cudaGetSymbolAddress((void **)&p, g_static_scratch));
        if (!p) return MD_ECUDA;
        ptr[dev] = p;
    }
    *out = ptr[dev];
    return MD_OK;
}

static bool static_on_device(const void *p)
{
    cudaPointerAttributes a;
    if (cudaPointerGetAttributes(&a, p) != cudaSuccess) {
        cudaGetLastError();
        return false;
    }
    return a.type == cudaMemoryTypeDevice || a.type == cudaMemoryTypeManaged;
}

extern "C" int md_forces_allpairs_static(const float *pos, int64_t N, double L, double rc, double eps, double sigma,
                                         int shifted, float *forces, double *pe_virial, void *cuda_stream)
{
    // argument checks first, before anything touches the device (the same rules as md_create)
    if (!pos || !forces || !pe_virial) return MD_EINVAL;
    if (!(N > 0) || !(L > 0.0) || !(rc > 0.0) || !(eps >= 0.0) || !(sigma > 0.0)) return MD_EINVAL;
    if (!isfinite(L) || !isfinite(rc) || !isfinite(eps) || !isfinite(sigma)) return MD_EINVAL;
    if (shifted < 0 || shifted > 2) return MD_EINVAL;
    if (N > MD_STATIC_MAX_ATOMS) return MD_EUNSUPPORTED;      // the scratch is sized for this many atoms
    const float Lf = (float)L;
    const double Ld = (double)Lf;                             // the box every path of the library uses (R13)
    if (rc > 0.5 * Ld) return MD_EINVAL;
    cudaStream_t st = (cudaStream_t)cuda_stream;

    double *scratch = nullptr;
    {
        const int r_ = static_scratch_ptr(&scratch);
        if (r_) return r_;
    }
    // nothing can be staged without allocating: all three arrays must already be in device memory
    if (!static_on_device(pos) || !static_on_device(forces) || !static_on_device(pe_virial)) return MD_EINVAL;

    PairParams P;
    memset(&P, 0, sizeof(P));
    P.rc = rc;
    P.rc2 = rc * rc;
    P.sig2 = sigma * sigma;
    P.eps24 = 24.0 * eps;
    P.eps4 = 4.0 * eps;
    const double s6 = pow(sigma * sigma / (rc * rc), 3.0);
    P.ushift = (shifted >= 1) ? 4.0 * eps * (s6 * s6 - s6) : 0.0;
    P.f_rc = (shifted == 2) ? 24.0 * eps * (2.0 * s6 * s6 - s6) / rc : 0.0;
    P.mode = shifted;
    P.kind = MD_POT_LJ;
    P.precise_r2 = 1.0e300;
    // FP32 accept threshold: rc^2 plus the worst rounding error of an FP32 r^2 from box-scale coordinates,
    // so that no pair inside rc in exact arithmetic is turned away before the FP64 decision
    const double errd = 4.0 * Ld * ldexp(1.0, -23);
    const double margin = 2.0 * sqrt(3.0) * (rc + errd) * errd + P.rc2 * 1e-6;
    P.rc2f_filter = nextafterf((float)(P.rc2 + margin), INFINITY);

    // j split: about SA_TARGET_BLOCKS blocks, chunks a multiple of 32 atoms
    const int n = (int)N;
    const int tiles = (n + SA_T - 1) / SA_T;
    int nsplit = (SA_TARGET_BLOCKS + tiles - 1) / tiles;
    const int max_split = (n + 31) / 32;
    if (nsplit > max_split) nsplit = max_split;
    int jchunk = (n + nsplit - 1) / nsplit;
    jchunk = (jchunk + 31) / 32 * 32;
    nsplit = (n + jchunk - 1) / jchunk;
    if ((int64_t)nsplit * 3 * n > SA_FPART_DOUBLES || tiles * nsplit > SA_MAX_BLOCKS || tiles > SA_MAX_TILES)
        return MD_EUNSUPPORTED;                               // cannot happen for N <= MD_STATIC_MAX_ATOMS

    CK(cudaMemsetAsync(scratch + SA_OFF_CTR, 0, SA_CTR_DOUBLES * sizeof(double), st));    // the arrival counters
    dim3 grid(tiles, nsplit);
    k_force_allpairs_static<<<grid, SA_T, 0, st>>>(pos, n, P, Lf, 1.0f / Lf, Ld, 1.0 / Ld, jchunk, scratch, forces,
                                                   pe_virial);
    CK(cudaGetLastError());
    CK(cudaStreamSynchronize(st));
    return MD_OK;
}
