// rand48 with O(log k) skip-ahead.
// PAPER.md:142-146 (Eq. 5): x <- (a x + c) mod 2^48, a = 0x5DEECE66D, c = 0xB, output from the
// new state's most-significant bits.  PAPER.md:150-162 (Eq. 6-7, sum bound corrected per R5):
// x_{n+m} = A_m x_n + C_m.  The paper leap-frogs S = 6144 threads over ONE stream after a
// serial warm-up; here every warp leap-frogs over a 128-draw window of its own segment of a
// stream, and reaches its start state by composing the maps (A_{2^b}, C_{2^b}) -- no serial
// warm-up, any number of streams, coalesced 16-byte stores of stream-major output.
#include "common.cuh"

#define R48_A 0x5DEECE66DULL
#define R48_C 0xBULL
#define R48_MASK 0xFFFFFFFFFFFFULL
#define R48_T 256
#define R48_TARGET_WARPS (148 * 64 * 4)

// The maps (A, C)_{2^b}, b < 48, in constant memory: every lane of a warp walks the bits of its skip distance in
// the same order, so each table read is one broadcast from the constant cache (they were global loads before).
__constant__ uint64_t g_r48_A[48];   // A_{2^b}
__constant__ uint64_t g_r48_C[48];   // C_{2^b}

// State after n further draws, by applying the power-of-two maps for the set bits of n.
__device__ __forceinline__ uint64_t r48_skip(uint64_t x, uint64_t n)
{
    n &= R48_MASK;                         // the period is 2^48
    for (int b = 0; n != 0; b++, n >>= 1)
        if (n & 1) x = (g_r48_A[b] * x + g_r48_C[b]) & R48_MASK;
    return x;
}

template <int KIND> struct R48Out;
template <> struct R48Out<0> { typedef uint32_t T; static __device__ __forceinline__ T cv(uint64_t x) { return (uint32_t)(x >> 16); } };
template <> struct R48Out<1> { typedef uint32_t T; static __device__ __forceinline__ T cv(uint64_t x) { return (uint32_t)(x >> 17); } };
template <> struct R48Out<2> {
    typedef double T;
    // x * 2^-48 exactly: 1.m with m = x << 4 is 1 + x 2^-48 in [1,2); subtracting 1 is exact.
    static __device__ __forceinline__ T cv(uint64_t x) { return __longlong_as_double((long long)(0x3FF0000000000000ULL | (x << 4))) - 1.0; }
};
template <> struct R48Out<3> { typedef uint64_t T; static __device__ __forceinline__ T cv(uint64_t x) { return x; } };

__device__ int g_r48_flag;           // set by a kernel that met a seed with bits above 47; read and cleared by the host

// One warp per (stream, segment).  Lane l keeps 4 states whose positions inside the current
// 128-draw window are pos[k]; every iteration applies (A_128, C_128) to all four.
template <int KIND>
__global__ void __launch_bounds__(R48_T)
k_rand48_fill(const uint64_t *__restrict__ seeds, int64_t nstreams, int64_t ndraws, int64_t seg, int64_t nseg,
              void *__restrict__ out_, int vec_ok)
{
    typedef typename R48Out<KIND>::T T;
    constexpr int V = 16 / sizeof(T);                  // draws per 16-byte vector: 4 or 2
    const int lane = threadIdx.x & 31;
    const int64_t gw = ((int64_t)blockIdx.x * R48_T + threadIdx.x) >> 5;
    if (gw >= nstreams * nseg) return;
    const int64_t s = gw / nseg, g = gw - s * nseg;
    const uint64_t seed = seeds[s];
    if (seed >> 48) {                                  // not a 48-bit state: the call fails (argument check, folded in)
        if (lane == 0) g_r48_flag = 1;
        return;
    }
    const int64_t start = g * seg;
    const int64_t len = min(seg, ndraws - start);
    T *out = (T *)out_ + (s * ndraws + start);

    const uint64_t A128 = g_r48_A[7], C128 = g_r48_C[7];
    uint64_t st[4];
    int pos[4];
    st[0] = r48_skip(seed, (uint64_t)(start + lane * V + 1));
    pos[0] = lane * V;
#pragma unroll
    for (int k = 1; k < V; k++) {
        st[k] = (R48_A * st[k - 1] + R48_C) & R48_MASK;
        pos[k] = pos[k - 1] + 1;
    }
    if (V == 2) {                                      // second vector: 64 draws further on
        const uint64_t A64 = g_r48_A[6], C64 = g_r48_C[6];
        st[2] = (A64 * st[0] + C64) & R48_MASK;
        st[3] = (A64 * st[1] + C64) & R48_MASK;
        pos[2] = pos[0] + 64;
        pos[3] = pos[1] + 64;
    }

    const int64_t nfull = vec_ok ? len / 128 : 0;
    for (int64_t it = 0; it < nfull; it++) {
        T *o = out + it * 128;
        if (V == 4) {
            uint4 v = make_uint4((uint32_t)R48Out<KIND>::cv(st[0]), (uint32_t)R48Out<KIND>::cv(st[1]),
                                 (uint32_t)R48Out<KIND>::cv(st[2]), (uint32_t)R48Out<KIND>::cv(st[3]));
            __stcs((uint4 *)(o + pos[0]), v);
        } else {
            T a0 = R48Out<KIND>::cv(st[0]), a1 = R48Out<KIND>::cv(st[1]);
            T a2 = R48Out<KIND>::cv(st[2]), a3 = R48Out<KIND>::cv(st[3]);
            ulonglong2 v0, v1;
            memcpy(&v0.x, &a0, 8); memcpy(&v0.y, &a1, 8);
            memcpy(&v1.x, &a2, 8); memcpy(&v1.y, &a3, 8);
            __stcs((ulonglong2 *)(o + pos[0]), v0);
            __stcs((ulonglong2 *)(o + pos[2]), v1);
        }
#pragma unroll
        for (int k = 0; k < 4; k++) st[k] = (A128 * st[k] + C128) & R48_MASK;
    }
    // scalar tail (and the whole segment when 16-byte stores are not aligned)
    for (int64_t base = nfull * 128; base < len; base += 128) {
#pragma unroll
        for (int k = 0; k < 4; k++) {
            if (base + pos[k] < len) out[base + pos[k]] = R48Out<KIND>::cv(st[k]);
            st[k] = (A128 * st[k] + C128) & R48_MASK;
        }
    }
}

// seeds[s] <- state after ndraws draws ("the thread saves the current state").
__global__ void __launch_bounds__(R48_T)
k_rand48_advance(uint64_t *__restrict__ seeds, int64_t nstreams, uint64_t ndraws)
{
    if (g_r48_flag) return;                            // the fill kernel refused a seed: no state moves
    int64_t s = (int64_t)blockIdx.x * R48_T + threadIdx.x;
    if (s < nstreams) seeds[s] = r48_skip(seeds[s], ndraws);
}

__global__ void __launch_bounds__(R48_T)
k_rand48_validate(const uint64_t *__restrict__ seeds, int64_t nstreams)
{
    int64_t s = (int64_t)blockIdx.x * R48_T + threadIdx.x;
    if (s < nstreams && (seeds[s] >> 48)) g_r48_flag = 1;
}

static cudaStream_t g_r48_stream = 0;
static int64_t g_r48_launches = 0;

// The skip-ahead table lives in __device__ memory, i.e. once per device: fill it on the first use on each
// device, and wait for it once, since later calls may come on other streams.
static int r48_ensure_table(cudaStream_t st)
{
    static bool ready[64] = {false};
    int dev = 0;
    CK(cudaGetDevice(&dev));
    if (dev < 0 || dev >= 64) return MD_EUNSUPPORTED;
    if (ready[dev]) return MD_OK;
    // (A, C)_{2^(b+1)} = (A, C)_{2^b} composed with itself: (A^2, A C + C)
    uint64_t hA[48], hC[48];
    uint64_t a = R48_A, c = R48_C;
    for (int b = 0; b < 48; b++) {
        hA[b] = a;
        hC[b] = c;
        c = (a * c + c) & R48_MASK;
        a = (a * a) & R48_MASK;
    }
    CK(cudaMemcpyToSymbolAsync(g_r48_A, hA, sizeof(hA), 0, cudaMemcpyHostToDevice, st));
    CK(cudaMemcpyToSymbolAsync(g_r48_C, hC, sizeof(hC), 0, cudaMemcpyHostToDevice, st));
    CK(cudaStreamSynchronize(st));                     // hA, hC are on the stack; later calls may use other streams
    ready[dev] = true;
    return MD_OK;
}

extern "C" int rand48_set_stream(void *stream)
{
    g_r48_stream = (cudaStream_t)stream;
    return MD_OK;
}

extern "C" int64_t rand48_kernel_launches(void) { return g_r48_launches; }

static bool on_device(const void *p)
{
    cudaPointerAttributes a;
    if (cudaPointerGetAttributes(&a, p) != cudaSuccess) {
        cudaGetLastError();
        return false;
    }
    return a.type == cudaMemoryTypeDevice || a.type == cudaMemoryTypeManaged;
}

extern "C" int rand48_fill(uint64_t *seeds, int64_t nstreams, int64_t ndraws, int kind, void *out)
{
    return rand48_fill_on(seeds, nstreams, ndraws, kind, out, (void *)g_r48_stream);
}

extern "C" int rand48_fill_on(uint64_t *seeds, int64_t nstreams, int64_t ndraws, int kind, void *out, void *stream)
{
    if (nstreams < 0 || ndraws < 0 || kind < 0 || kind > 3) return MD_EINVAL;
    if (nstreams == 0) return MD_OK;
    if (!seeds) return MD_EINVAL;
    if (ndraws > 0 && !out) return MD_EINVAL;
    if (ndraws > (int64_t)R48_MASK) return MD_EINVAL;
    cudaStream_t st = (cudaStream_t)stream;
    const size_t esize = (kind <= 1) ? 4 : 8;
    const bool seeds_dev = on_device(seeds);
    const bool out_dev = ndraws == 0 || on_device(out);
    uint64_t *dseeds = seeds;
    void *dout = out;
    int rc = MD_OK;

    // seeds must be 48-bit states (argument check): on the host for host arrays.  For device arrays the fill kernel
    // itself checks the seed it reads (a warp that meets a bad one stores nothing and raises g_r48_flag, the advance
    // kernel then leaves every state alone) and the flag comes back with the synchronisation that ends the call:
    // no separate validation pass, copy and synchronisation in front of the fill.  On MD_EINVAL the seeds are
    // unchanged and the contents of `out` are unspecified.  Only a call with nothing to draw validates by itself.
    if (seeds_dev && ndraws == 0) {
        int flag = 0;
        k_rand48_validate<<<(unsigned)((nstreams + R48_T - 1) / R48_T), R48_T, 0, st>>>(seeds, nstreams);
        CK(cudaGetLastError());
        g_r48_launches++;
        CK(cudaMemcpyFromSymbolAsync(&flag, g_r48_flag, sizeof(int), 0, cudaMemcpyDeviceToHost, st));
        CK(cudaStreamSynchronize(st));
        if (flag) {
            const int zero = 0;
            CK(cudaMemcpyToSymbol(g_r48_flag, &zero, sizeof(int)));
            return MD_EINVAL;
        }
    } else if (!seeds_dev) {
        for (int64_t i = 0; i < nstreams; i++)
            if (seeds[i] >> 48) return MD_EINVAL;
    }
    if (ndraws == 0) return MD_OK;

    {
        const int r_ = r48_ensure_table(st);
        if (r_) return r_;
    }
    if (!seeds_dev) {
        dseeds = (uint64_t *)ljmd_dev_alloc(nstreams * 8, st);
        if (!dseeds) return MD_ENOMEM;
        cudaError_t e = cudaMemcpyAsync(dseeds, seeds, (size_t)nstreams * 8, cudaMemcpyHostToDevice, st);
        if (e != cudaSuccess) { ljmd_note_cuda_error(e, "seed upload", __FILE__, __LINE__); rc = MD_ECUDA; goto done; }
    }
    if (!out_dev) {
        dout = ljmd_dev_alloc((int64_t)((size_t)nstreams * ndraws * esize), st);
        if (!dout) { rc = MD_ENOMEM; goto done; }
    }
    {
        // segment length: a multiple of 128 draws, at least 1024, sized for about four waves of resident warps
        // (148 SMs x 64): a warp pays its skip-ahead (one table step per set bit of its start, up to 28 for the
        // 2^28-draw stream) once per segment, so few long segments beat many short ones
        int64_t total = nstreams * ndraws;
        int64_t seg = (total / R48_TARGET_WARPS + 127) / 128 * 128;
        if (seg < 1024) seg = 1024;
        int64_t nd128 = (ndraws + 127) / 128 * 128;
        if (seg > nd128) seg = nd128;
        int64_t nseg = (ndraws + seg - 1) / seg;
        int64_t nwarps = nstreams * nseg;
        int64_t nblocks = (nwarps * 32 + R48_T - 1) / R48_T;
        if (nblocks > 0x7FFFFFFF) { rc = MD_EUNSUPPORTED; goto done; }
        int vec_ok = (((uintptr_t)dout) % 16 == 0) && ((ndraws * esize) % 16 == 0);
        switch (kind) {
        case 0: k_rand48_fill<0><<<(unsigned)nblocks, R48_T, 0, st>>>(dseeds, nstreams, ndraws, seg, nseg, dout, vec_ok); break;
        case 1: k_rand48_fill<1><<<(unsigned)nblocks, R48_T, 0, st>>>(dseeds, nstreams, ndraws, seg, nseg, dout, vec_ok); break;
        case 2: k_rand48_fill<2><<<(unsigned)nblocks, R48_T, 0, st>>>(dseeds, nstreams, ndraws, seg, nseg, dout, vec_ok); break;
        default: k_rand48_fill<3><<<(unsigned)nblocks, R48_T, 0, st>>>(dseeds, nstreams, ndraws, seg, nseg, dout, vec_ok); break;
        }
        cudaError_t e = cudaGetLastError();
        if (e != cudaSuccess) { ljmd_note_cuda_error(e, "k_rand48_fill", __FILE__, __LINE__); rc = MD_ECUDA; goto done; }
        g_r48_launches++;
        k_rand48_advance<<<(unsigned)((nstreams + R48_T - 1) / R48_T), R48_T, 0, st>>>(dseeds, nstreams, (uint64_t)ndraws);
        e = cudaGetLastError();
        if (e != cudaSuccess) { ljmd_note_cuda_error(e, "k_rand48_advance", __FILE__, __LINE__); rc = MD_ECUDA; goto done; }
        g_r48_launches++;
        if (!out_dev) {
            e = cudaMemcpyAsync(out, dout, (size_t)nstreams * ndraws * esize, cudaMemcpyDeviceToHost, st);
            if (e != cudaSuccess) { ljmd_note_cuda_error(e, "output download", __FILE__, __LINE__); rc = MD_ECUDA; goto done; }
        }
        if (!seeds_dev) {
            e = cudaMemcpyAsync(seeds, dseeds, (size_t)nstreams * 8, cudaMemcpyDeviceToHost, st);
            if (e != cudaSuccess) { ljmd_note_cuda_error(e, "seed download", __FILE__, __LINE__); rc = MD_ECUDA; goto done; }
        }
        int flag = 0;
        if (seeds_dev) {
            e = cudaMemcpyFromSymbolAsync(&flag, g_r48_flag, sizeof(int), 0, cudaMemcpyDeviceToHost, st);
            if (e != cudaSuccess) { ljmd_note_cuda_error(e, "seed flag", __FILE__, __LINE__); rc = MD_ECUDA; goto done; }
        }
        e = cudaStreamSynchronize(st);
        if (e != cudaSuccess) { ljmd_note_cuda_error(e, "rand48_fill sync", __FILE__, __LINE__); rc = MD_ECUDA; }
        else if (flag) {
            const int zero = 0;
            cudaMemcpyToSymbol(g_r48_flag, &zero, sizeof(int));
            rc = MD_EINVAL;
        }
    }
done:
    if (!seeds_dev && dseeds) { cudaStreamSynchronize(st); ljmd_dev_free(dseeds, st); }
    if (!out_dev && dout && dout != out) { cudaStreamSynchronize(st); ljmd_dev_free(dout, st); }
    return rc;
}

// ---------------------------------------------------------------------------------------
// Maxwell-Boltzmann start velocities on the device (first half): the rand48 draws
// are consumed in registers instead of being stored to HBM (PAPER.md:176-178 names that store as the
// cost of the generator).  Atom `id` owns draws 6 id .. 6 id + 5 of ONE stream and reaches them by
// skip-ahead; per component u1, u2 -> v = sqrt(T) sqrt(-2 ln(1 - u1)) cos(2 pi u2) in FP64; then the
// mean is removed and the set rescaled to sum v^2 = 3 N T (R11).  Same recipe as oracle mb_velocities.
#define MB_T 256

__global__ void __launch_bounds__(MB_T)
k_mb_draw(const float4 *__restrict__ pos, int64_t N, uint64_t x0, double sqrtT, double *__restrict__ vraw,
          double *__restrict__ part)                                    // part: [4][gridDim.x] sums of vx, vy, vz, v^2
{
    __shared__ double red[32];
    const int64_t slot = (int64_t)blockIdx.x * MB_T + threadIdx.x;
    double v[3] = {0.0, 0.0, 0.0};
    if (slot < N) {
        const uint64_t id = (uint64_t)__float_as_int(pos[slot].w);         // caller's atom index
        uint64_t x = r48_skip(x0, 6ull * id);
#pragma unroll
        for (int c = 0; c < 3; c++) {
            x = (R48_A * x + R48_C) & R48_MASK;
            const double u1 = R48Out<2>::cv(x);
            x = (R48_A * x + R48_C) & R48_MASK;
            const double u2 = R48Out<2>::cv(x);
            v[c] = sqrtT * sqrt(-2.0 * log(1.0 - u1)) * cos(6.283185307179586476925286766559 * u2);
            vraw[3 * slot + c] = v[c];
        }
    }
    const double q[4] = {v[0], v[1], v[2], v[0] * v[0] + v[1] * v[1] + v[2] * v[2]};
#pragma unroll
    for (int k = 0; k < 4; k++) {
        const double t = block_sum(q[k], red);
        if (threadIdx.x == 0) part[(size_t)k * gridDim.x + blockIdx.x] = t;
    }
}

// mean[3] and scale from the block partials: sum (v - m)^2 = sum v^2 - N m^2.  One block.
__global__ void __launch_bounds__(1024)
k_mb_moments(const double *__restrict__ part, int nblocks, int64_t N, double T, double *__restrict__ mom)
{
    __shared__ double red[32];
    __shared__ double tot[4];
    for (int k = 0; k < 4; k++) {
        double a = 0.0;
        for (int i = threadIdx.x; i < nblocks; i += blockDim.x) a += part[(size_t)k * nblocks + i];
        a = block_sum(a, red);
        if (threadIdx.x == 0) tot[k] = a;
        __syncthreads();
    }
    if (threadIdx.x == 0) {
        const double n = (double)N;
        const double mx = tot[0] / n, my = tot[1] / n, mz = tot[2] / n;
        const double s2 = tot[3] - n * (mx * mx + my * my + mz * mz);
        mom[0] = mx; mom[1] = my; mom[2] = mz;
        mom[3] = sqrt(3.0 * n * T / s2);
    }
}

__global__ void __launch_bounds__(MB_T)
k_mb_apply(float4 *__restrict__ vel, const double *__restrict__ vraw, const double *__restrict__ mom, int64_t N)
{
    const int64_t slot = (int64_t)blockIdx.x * MB_T + threadIdx.x;
    if (slot >= N) return;
    const double sc = mom[3];
    vel[slot] = make_float4((float)((vraw[3 * slot] - mom[0]) * sc), (float)((vraw[3 * slot + 1] - mom[1]) * sc),
                            (float)((vraw[3 * slot + 2] - mom[2]) * sc), 0.f);
}

// vraw: [3 N] doubles, part: [4 * nblocks] doubles, mom: [4] doubles (device scratch of the caller)
int ljmd_mb_velocities(md_sim *s, double T, uint64_t seed48, double *vraw, double *part, double *mom)
{
    cudaStream_t st = s->stream;
    {
        const int r_ = r48_ensure_table(st);
        if (r_) return r_;
    }
    const int nb = (int)((s->N + MB_T - 1) / MB_T);
    k_mb_draw<<<nb, MB_T, 0, st>>>(s->pos, s->N, seed48, sqrt(T), vraw, part);
    CKL(s);
    k_mb_moments<<<1, 1024, 0, st>>>(part, nb, s->N, T, mom);
    CKL(s);
    k_mb_apply<<<nb, MB_T, 0, st>>>(s->vel, vraw, mom, s->N);
    CKL(s);
    return MD_OK;
}

// ---------------------------------------------------------------------------------------
// Second half-kick + Andersen thermostat + KE (second half; reading R24 of DESIGN.md,
// same draw ownership as oracle andersen_collide): after the half-kick of step t atom `id` takes the 7
// draws starting at 7 (t N + id) of one rand48 stream, reached by skip-ahead and consumed in registers;
// collision iff the 32 high bits of the first are < thr; the new velocity is computed in FP64.
__global__ void __launch_bounds__(MB_T)
k_kick_andersen(float4 *__restrict__ vel, const float4 *__restrict__ frc, const float4 *__restrict__ pos, int64_t N,
                float hdt, double sqrtT, uint32_t thr, uint64_t seed, const uint64_t *__restrict__ tptr,
                double *__restrict__ part_ke)
{
    __shared__ double red[32];
    const uint64_t t = *tptr;                            // step index, in device memory: the launch can sit in a graph
    const int64_t slot = (int64_t)blockIdx.x * MB_T + threadIdx.x;
    double ke = 0.0;
    if (slot < N) {
        float4 v = vel[slot];
        const float4 f = frc[slot];
        v.x = fmaf(hdt, f.x, v.x);
        v.y = fmaf(hdt, f.y, v.y);
        v.z = fmaf(hdt, f.z, v.z);
        const uint64_t id = (uint64_t)__float_as_int(pos[slot].w);
        uint64_t x = r48_skip(seed, 7ull * (t * (uint64_t)N + id));
        x = (R48_A * x + R48_C) & R48_MASK;
        if ((uint32_t)(x >> 16) < thr) {
            double nv[3];
#pragma unroll
            for (int c = 0; c < 3; c++) {
                x = (R48_A * x + R48_C) & R48_MASK;
                const double u1 = R48Out<2>::cv(x);
                x = (R48_A * x + R48_C) & R48_MASK;
                const double u2 = R48Out<2>::cv(x);
                nv[c] = sqrtT * sqrt(-2.0 * log(1.0 - u1)) * cos(6.283185307179586476925286766559 * u2);
            }
            v.x = (float)nv[0]; v.y = (float)nv[1]; v.z = (float)nv[2];
        }
        vel[slot] = v;
        ke = 0.5 * ((double)v.x * v.x + (double)v.y * v.y + (double)v.z * v.z);
    }
    ke = block_sum(ke, red);
    if (threadIdx.x == 0) part_ke[blockIdx.x] = ke;
}

__global__ void __launch_bounds__(1) k_andersen_tick(uint64_t *t) { *t += 1ull; }

int ljmd_kick_andersen(md_sim *s)
{
    cudaStream_t st = s->stream;
    {
        const int r_ = r48_ensure_table(st);
        if (r_) return r_;
    }
    const int nb = (int)((s->N + MB_T - 1) / MB_T);
    k_kick_andersen<<<nb, MB_T, 0, st>>>(s->vel, s->frc, s->pos, s->N, s->hdtf, sqrt(s->and_T), s->and_thr, s->and_seed,
                                         s->and_t_dev, s->part);
    CKL(s);
    k_andersen_tick<<<1, 1, 0, st>>>(s->and_t_dev);
    CKL(s);
    s->n_ke = nb;
    s->and_t++;
    return MD_OK;
}
