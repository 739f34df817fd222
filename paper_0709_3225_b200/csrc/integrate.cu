// Velocity-Verlet integration kernels (step order per DESIGN.md R4), state
// packing, and the KE/PE/virial reductions.
// All are HBM-streaming kernels: one float4 per atom per array, 16-byte vector accesses.
#include "common.cuh"

#define IT 256   // threads per block for the streaming kernels

// General wrap for md_set_state (positions may be any finite value).
__device__ __forceinline__ float wrap_any(float x, float L)
{
    x -= L * floorf(x / L);
    if (x >= L || x < 0.0f) x = 0.0f;
    return x;
}

__global__ void __launch_bounds__(IT)
k_pack_state(float4 *__restrict__ pos, float4 *__restrict__ vel, const float *__restrict__ in_pos,
             const float *__restrict__ in_vel, int64_t N, float L)
{
    int64_t i = (int64_t)blockIdx.x * IT + threadIdx.x;
    if (i >= N) return;
    float4 p, v;
    p.x = wrap_any(in_pos[3 * i + 0], L);
    p.y = wrap_any(in_pos[3 * i + 1], L);
    p.z = wrap_any(in_pos[3 * i + 2], L);
    p.w = __int_as_float((int)i);
    v.x = in_vel[3 * i + 0];
    v.y = in_vel[3 * i + 1];
    v.z = in_vel[3 * i + 2];
    v.w = 0.0f;
    pos[i] = p;
    vel[i] = v;
}

// out[id][0..2] = src[slot].xyz where id is carried in pos[slot].w
__global__ void __launch_bounds__(IT)
k_unpack(float *__restrict__ out, const float4 *__restrict__ src, const float4 *__restrict__ pos, int64_t N)
{
    int64_t i = (int64_t)blockIdx.x * IT + threadIdx.x;
    if (i >= N) return;
    float4 a = src[i];
    int64_t id = __float_as_int(pos[i].w);
    out[3 * id + 0] = a.x;
    out[3 * id + 1] = a.y;
    out[3 * id + 2] = a.z;
}

// a1: v += (dt/2) F;  x += dt v;  wrap.  KICKS = 2 also applies the second half-kick that the
// previous step of the same md_step call left pending (same F, two separate FMAs, so the
// velocities are bit-identical to the unfused sequence).
template <int KICKS>
__global__ void __launch_bounds__(IT)
k_kick_drift(float4 *__restrict__ pos, float4 *__restrict__ vel, const float4 *__restrict__ frc,
             int64_t N, float hdt, float dt, float L)
{
    int64_t i = (int64_t)blockIdx.x * IT + threadIdx.x;
    if (i >= N) return;
    float4 p = pos[i], v = vel[i], f = frc[i];
#pragma unroll
    for (int k = 0; k < KICKS; k++) {
        v.x = fmaf(hdt, f.x, v.x);
        v.y = fmaf(hdt, f.y, v.y);
        v.z = fmaf(hdt, f.z, v.z);
    }
    p.x = wrap_drift(fmaf(dt, v.x, p.x), L);
    p.y = wrap_drift(fmaf(dt, v.y, p.y), L);
    p.z = wrap_drift(fmaf(dt, v.z, p.z), L);
    pos[i] = p;
    vel[i] = v;
}

// a5: v += (dt/2) F;  KE partial = (1/2) sum v^2 per block (FP64 accumulation).
template <bool KICK>
__global__ void __launch_bounds__(IT)
k_kick_ke(float4 *__restrict__ vel, const float4 *__restrict__ frc, int64_t N, float hdt,
          double *__restrict__ part_ke)
{
    __shared__ double sm[32];
    int64_t i = (int64_t)blockIdx.x * IT + threadIdx.x;
    double ke = 0.0;
    if (i < N) {
        float4 v = vel[i];
        if (KICK) {
            float4 f = frc[i];
            v.x = fmaf(hdt, f.x, v.x);
            v.y = fmaf(hdt, f.y, v.y);
            v.z = fmaf(hdt, f.z, v.z);
            vel[i] = v;
        }
        ke = 0.5 * ((double)v.x * v.x + (double)v.y * v.y + (double)v.z * v.z);
    }
    ke = block_sum(ke, sm);
    if (threadIdx.x == 0) part_ke[blockIdx.x] = ke;
}

// a6: deterministic second pass: energies[k] = sum of part[k][0..n_k) for k = KE, PE, W.
__global__ void __launch_bounds__(1024)
k_reduce_energies(const double *__restrict__ part, int cap, int n_ke, int n_pe, double *__restrict__ energies)
{
    __shared__ double sm[32];
    int k = blockIdx.x;                       // 0 KE, 1 PE, 2 W
    int n = (k == 0) ? n_ke : n_pe;
    const double *p = part + (size_t)k * cap;
    double acc = 0.0;
    for (int i = threadIdx.x; i < n; i += blockDim.x) acc += p[i];
    acc = block_sum(acc, sm);
    if (threadIdx.x == 0) energies[k] = acc;
}

static inline int nblk(int64_t N) { return (int)((N + IT - 1) / IT); }

int ljmd_pack_state(md_sim *s, const float *dpos, const float *dvel)
{
    k_pack_state<<<nblk(s->N), IT, 0, s->stream>>>(s->pos, s->vel, dpos, dvel, s->N, s->Lf);
    CKL(s);
    return MD_OK;
}

int ljmd_unpack(md_sim *s, const float4 *src, float *dout)
{
    k_unpack<<<nblk(s->N), IT, 0, s->stream>>>(dout, src, s->pos, s->N);
    CKL(s);
    return MD_OK;
}

int ljmd_kick_drift(md_sim *s, int kicks)
{
    if (kicks == 2)
        k_kick_drift<2><<<nblk(s->N), IT, 0, s->stream>>>(s->pos, s->vel, s->frc, s->N, s->hdtf, s->dtf, s->Lf);
    else
        k_kick_drift<1><<<nblk(s->N), IT, 0, s->stream>>>(s->pos, s->vel, s->frc, s->N, s->hdtf, s->dtf, s->Lf);
    CKL(s);
    return MD_OK;
}

int ljmd_kick_ke(md_sim *s)
{
    k_kick_ke<true><<<nblk(s->N), IT, 0, s->stream>>>(s->vel, s->frc, s->N, s->hdtf, s->part);
    CKL(s);
    s->n_ke = nblk(s->N);
    return MD_OK;
}

int ljmd_ke_only(md_sim *s)
{
    k_kick_ke<false><<<nblk(s->N), IT, 0, s->stream>>>(s->vel, s->frc, s->N, 0.0f, s->part);
    CKL(s);
    s->n_ke = nblk(s->N);
    return MD_OK;
}

int ljmd_reduce_energies(md_sim *s)
{
    k_reduce_energies<<<3, 1024, 0, s->stream>>>(s->part, s->part_cap, s->n_ke, s->n_pe, s->energies);
    CKL(s);
    return MD_OK;
}
