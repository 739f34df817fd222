// All-pairs O(N^2) Lennard-Jones force under minimum image.
// PAPER.md:49-52 (Eq. 1) and :70-76 (Sec. 2.1): one thread per atom i, the j atoms staged
// through shared memory in tiles shared by the block.  What differs from the paper's G80
// kernel is listed in DESIGN.md section 7: the inner loop is an FP32 distance *filter* (only
// ~0.16 % of pairs are inside rc at N = 32000), accepted pairs are re-evaluated exactly in
// FP64 from the original coordinates, the j range is split across blockIdx.y so small N still
// fills 148 SMs, and partial forces are combined in a deterministic second pass.
#include "common.cuh"
#include "pair.cuh"

#define AP_T 128

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

int ljmd_forces_allpairs(md_sim *s)
{
    int N = (int)s->N;
    int niblk = (N + AP_T - 1) / AP_T;
    int nsplit = s->ap_nsplit;
    int jchunk = (N + nsplit - 1) / nsplit;
    jchunk = ((jchunk + AP_T - 1) / AP_T) * AP_T;
    dim3 grid(niblk, nsplit);
    double *ppe = s->part + (size_t)s->part_cap;
    double *pw = s->part + 2 * (size_t)s->part_cap;
    k_force_allpairs_general<<<grid, AP_T, 0, s->stream>>>(
        s->pos, N, s->pp, s->Lf, 1.0f / s->Lf, s->L, 1.0 / s->L, jchunk, s->fpart, ppe, pw);
    CKL(s);
    ljmd_tick(s, TAG_FORCE);
    s->n_pe = niblk * nsplit;
    k_combine_forces<<<(N + 255) / 256, 256, 0, s->stream>>>(s->frc, s->fpart, N, nsplit);
    CKL(s);
    ljmd_tick(s, TAG_OTHER);
    return MD_OK;
}
