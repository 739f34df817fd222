// Neighbour lists built from the cell list and reused over several steps (the
// paper discusses Verlet lists with a skin in PAPER.md:100-104 and keeps the cell list; here they are
// a third force path, algo = MD_VERLET, on top of the same counting sort).
//   * cells of side >= rc + skin; the list of atom i holds every j with r < rc + skin at build time;
//   * between builds atoms stay in their slot and keep their "home" cell; the integrator recomputes the
//     cell-local coordinate l = x - origin(home cell) from the wrapped position every step (exact, or
//     within 1.2e-7 next to the box origin, like the cell path: DESIGN.md section 5), so the stored
//     position stays the single source of truth and the oracle sees exactly what the kernels use;
//   * a list is valid while no atom has moved more than skin / 2 since the build: the integrator takes
//     the maximum squared displacement with one atomicMax per block, a one-thread kernel turns it into
//     a rebuild flag, and the build kernels (histogram, scan, scatter, copy-back, list) are launched
//     every step and return at once when the flag is clear - no host round trip, graph-replayable;
//   * list entry = slot of j (23 bits) | index (7 bits) into a table of the 125 possible offsets
//     between the origins of two neighbouring home cells ({0, +-side, +-last} per dimension, exact);
//   * force kernel: one thread per atom walks its list (transposed layout, coalesced), FP32 pair term
//     outside the steep part, close and near-cutoff pairs queued and evaluated in FP64 from the exact
//     local coordinates (same split as the cell path).
#include <math.h>
#include "common.cuh"
#include "pair.cuh"

#ifndef VL_T
#define VL_T 128                      // threads per block of the list and force kernels
#endif
#ifndef VL_Q
#define VL_Q 10                       // queued FP64 pairs per thread
#endif
#ifndef VL_U
#define VL_U 4                        // list entries (gathers) in flight per thread
#endif
#ifndef VL_MINB
#define VL_MINB 8
#endif
#define VL_JMASK 0x7fffffu
#define VL_CELLMASK 0x3fffffff
#define VL_INERT (31u << 23)            // offset index 31 = (+side, +side, +side): beyond any cutoff

// offset code of one dimension: 0: same cell, 1: +side, 2: -side, 3: +last, 4: -last
__device__ __forceinline__ float vl_code_value(int code, const Grid &g)
{
    return code == 0 ? 0.f : code == 1 ? g.side : code == 2 ? -g.side : code == 3 ? g.last : -g.last;
}

// cell-local coordinate of the wrapped position x for home cell index c (one dimension).  Exact in every case
// but one: home cell near the top of the box and the atom wrapped to x ~ 0, where x has bits below the 2^-22
// grid of l = x + (L - o).  There the stored position is moved onto that grid (by <= 1.2e-7, less than the
// rounding the drift x + dt v has near the top of the box anyway), so that the local coordinate the force
// kernels see and the position the caller reads back stay the same point: without it the forces of such an
// atom are those of a point up to 1.2e-7 away, 2e-5 off on a close pair (measured at N = 2,048,000).
__device__ __forceinline__ float vl_local(float &x, int c, const Grid &g)
{
    const float o = (float)c * g.side;                  // exact
    float l = x - o;                                    // exact unless the atom crossed the periodic seam
    if (l > 0.5f * g.L) l = (x - g.L) - o;              // home cell near 0, atom wrapped to the top: x - L is exact
    else if (l < -0.5f * g.L) {                         // home cell near the top, atom wrapped to x ~ 0
        const float C = g.L - o;                        // exact
        l = x + C;
        x = l - C;                                      // exact, >= 0
    }
    return l;
}

__global__ void __launch_bounds__(1) k_vl_decide(VlCtl *ctl, unsigned thr_bits)
{
    const unsigned m = ctl->maxd2;
    const int asked = ctl->force;                        // set by the host only (vl_force_build)
    const int rb = (m > thr_bits || asked) ? 1 : 0;
    ctl->rebuild = rb;
    ctl->force = 0;
    ctl->maxd2 = 0u;
    if (rb) {
        ctl->nbuilds++;
        // `overflow` is sticky across the builds the device decides on its own: md_step reads it once, after all
        // steps, and a list truncated in the middle of the run must still be reported even if a later build
        // fitted.  Only a build the host asked for (after md_set_state, a grow, another path) starts afresh.
        if (asked) ctl->overflow = 0;
    }
    ctl->nsteps++;
}

// [pending half-kick,] half-kick, drift, wrap (same arithmetic as k_kick_drift), then the local
// coordinate in the home cell and the squared displacement since the last build.
template <int KICKS>
__global__ void __launch_bounds__(256)
k_vl_kick_drift(float4 *__restrict__ pos, float4 *__restrict__ vel, const float4 *__restrict__ frc,
                float4 *__restrict__ lpos, const float4 *__restrict__ lbuild, int N, float hdt, float dt, Grid g,
                VlCtl *__restrict__ ctl)
{
    const int i = blockIdx.x * 256 + threadIdx.x;
    float d2 = 0.f;
    if (i < N) {
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
        vel[i] = v;
        float4 l = lpos[i];
        const float4 l0 = lbuild[i];
        const int c = __float_as_int(l.w) & VL_CELLMASK;
        const int cz = c % g.n, cy = (c / g.n) % g.n, cx = c / (g.n * g.n);
        l.x = vl_local(p.x, cx, g);
        l.y = vl_local(p.y, cy, g);
        l.z = vl_local(p.z, cz, g);
        pos[i] = p;
        lpos[i] = l;
        const float ex = l.x - l0.x, ey = l.y - l0.y, ez = l.z - l0.z;
        d2 = fmaf(ex, ex, fmaf(ey, ey, ez * ez));
    }
    d2 = fmaxf(d2, __shfl_xor_sync(0xffffffffu, d2, 16));
    d2 = fmaxf(d2, __shfl_xor_sync(0xffffffffu, d2, 8));
    d2 = fmaxf(d2, __shfl_xor_sync(0xffffffffu, d2, 4));
    d2 = fmaxf(d2, __shfl_xor_sync(0xffffffffu, d2, 2));
    d2 = fmaxf(d2, __shfl_xor_sync(0xffffffffu, d2, 1));
    if ((threadIdx.x & 31) == 0 && d2 > 0.f) atomicMax(&ctl->maxd2, __float_as_uint(d2));   // positive floats order as unsigned
}

__device__ __forceinline__ int vl_cell_coord(float x, const Grid &g)
{
    int c = min((int)(x * g.inv_side), g.n - 1);
    const float o = (float)c * g.side;
    if (x < o) c--;
    else if (c < g.n - 1 && x >= o + g.side) c++;
    return c;
}

__global__ void __launch_bounds__(256)
k_vl_bin(const float4 *__restrict__ pos, int N, Grid g, int *__restrict__ cell_of, int *__restrict__ rank,
         int *__restrict__ cell_count, const VlCtl *__restrict__ ctl)
{
    if (!ctl->rebuild) return;
    for (int i = blockIdx.x * 256 + threadIdx.x; i < N; i += gridDim.x * 256) {      // small grid: cheap when idle
        const float4 p = pos[i];
        const int c = (vl_cell_coord(p.x, g) * g.n + vl_cell_coord(p.y, g)) * g.n + vl_cell_coord(p.z, g);
        cell_of[i] = c;
        rank[i] = atomicAdd(&cell_count[c], 1);
    }
}

// Scatter into cell order (to the spare buffers), with the cell-local coordinates.
__global__ void __launch_bounds__(256)
k_vl_scatter(const float4 *__restrict__ pos, const float4 *__restrict__ vel, int N, Grid g,
             const int *__restrict__ cell_of, const int *__restrict__ rank, const int *__restrict__ cell_start,
             float4 *__restrict__ pos2, float4 *__restrict__ vel2, float4 *__restrict__ lpos,
             const VlCtl *__restrict__ ctl)
{
    if (!ctl->rebuild) return;
    for (int i = blockIdx.x * 256 + threadIdx.x; i < N; i += gridDim.x * 256) {
        const int c = cell_of[i];
        const int dst = cell_start[c] + rank[i];
        const float4 p = pos[i];
        const int cz = c % g.n, cy = (c / g.n) % g.n, cx = c / (g.n * g.n);
        float4 l;
        l.x = p.x - (float)cx * g.side;                    // exact
        l.y = p.y - (float)cy * g.side;
        l.z = p.z - (float)cz * g.side;
        l.w = __int_as_float(c);
        pos2[dst] = p;
        vel2[dst] = vel[i];
        lpos[dst] = l;
    }
}

// The host never swaps buffers on this path (it does not know whether a build happened): copy back.
__global__ void __launch_bounds__(256)
k_vl_copyback(float4 *__restrict__ pos, float4 *__restrict__ vel, float4 *__restrict__ lbuild,
              const float4 *__restrict__ pos2, const float4 *__restrict__ vel2, const float4 *__restrict__ lpos, int N,
              const VlCtl *__restrict__ ctl)
{
    if (!ctl->rebuild) return;
    for (int i = blockIdx.x * 256 + threadIdx.x; i < N; i += gridDim.x * 256) {
        pos[i] = pos2[i];
        vel[i] = vel2[i];
        lbuild[i] = lpos[i];
    }
}

// Neighbour list of every atom from the 27 cells around its home cell: r < rc + skin in exact
// local coordinates.  list[k * npad + i] = slot of j | offset-table index << 23.
__global__ void __launch_bounds__(VL_T)
k_vl_build(const float4 *__restrict__ lpos, const int *__restrict__ cell_start, int N, int npad, Grid g, float rl2,
           int cap, unsigned *__restrict__ list, int *__restrict__ count, VlCtl *__restrict__ ctl, int half)
{
    if (!ctl->rebuild) return;
    const int i = blockIdx.x * VL_T + threadIdx.x;
    if (i >= N) return;
    const float4 li = lpos[i];
    const int c = __float_as_int(li.w) & VL_CELLMASK, n = g.n;
    const int cz = c % n, cy = (c / n) % n, cx = c / (n * n);
    int cnt = 0;
    for (int ax = -1; ax <= 1; ax++) {
        int nx = cx + ax;
        nx += (nx < 0) ? n : 0; nx -= (nx >= n) ? n : 0;
        const int kx = (ax == 0) ? 0 : (ax > 0 ? ((cx == n - 1) ? 3 : 1) : ((nx == n - 1) ? 4 : 2));
        const float ox = vl_code_value(kx, g);
        for (int ay = -1; ay <= 1; ay++) {
            int ny = cy + ay;
            ny += (ny < 0) ? n : 0; ny -= (ny >= n) ? n : 0;
            const int ky = (ay == 0) ? 0 : (ay > 0 ? ((cy == n - 1) ? 3 : 1) : ((ny == n - 1) ? 4 : 2));
            const float oy = vl_code_value(ky, g);
            for (int az = -1; az <= 1; az++) {
                int nz = cz + az;
                nz += (nz < 0) ? n : 0; nz -= (nz >= n) ? n : 0;
                const int kz = (az == 0) ? 0 : (az > 0 ? ((cz == n - 1) ? 3 : 1) : ((nz == n - 1) ? 4 : 2));
                const float oz = vl_code_value(kz, g);
                const unsigned tag = (unsigned)(kx + 5 * ky + 25 * kz) << 23;
                const int nb = (nx * n + ny) * n + nz;
                const int jb = cell_start[nb], je = cell_start[nb + 1];
                for (int j = jb; j < je; j++) {
                    const float4 lj = lpos[j];
                    const float dx = (lj.x - li.x) + ox, dy = (lj.y - li.y) + oy, dz = (lj.z - li.z) + oz;
                    const float r2 = fmaf(dx, dx, fmaf(dy, dy, dz * dz));
                    if (r2 < rl2 && j != i && (!half || j > i)) {      // half lists: each pair once, in the lower slot's list
                        if (cnt < cap) list[(size_t)cnt * npad + i] = (unsigned)j | tag;
                        cnt++;
                    }
                }
            }
        }
    }
    if (cnt > cap) atomicMax(&ctl->overflow, cnt);         // the length this list needs
    cnt = min(cnt, cap);
    // pad to a multiple of VL_U with inert entries: the atom itself, displaced by a cell diagonal
    for (; cnt % VL_U; cnt++) list[(size_t)cnt * npad + i] = (unsigned)i | VL_INERT;
    count[i] = cnt;
}

struct VlConst {
    float rc2_lo, rc2_hi, p2, sig2, eps24, eps48;
};

// FP64 pair term from the exact local coordinates of i and of list entry e
__device__ __forceinline__ void vl_precise(const float4 *__restrict__ lpos, const float4 *offt, const PairParams &P,
                                           const float4 &li, unsigned e, double &fx, double &fy, double &fz,
                                           double &pe, double &w)
{
    const float4 lj = lpos[e & VL_JMASK];
    const float4 o = offt[e >> 23];
    const double ex = ((double)lj.x - (double)li.x) + (double)o.x;
    const double ey = ((double)lj.y - (double)li.y) + (double)o.y;
    const double ez = ((double)lj.z - (double)li.z) + (double)o.z;
    pair_f64(P, ex, ey, ez, fx, fy, fz, pe, w);
}

// reaction force of one pair on atom j: one vector reduction into the L2 (no return value)
__device__ __forceinline__ void vl_react(float4 *frc, int j, float x, float y, float z)
{
    asm volatile("red.global.add.v4.f32 [%0], {%1, %2, %3, %4};" :: "l"(frc + j), "f"(x), "f"(y), "f"(z), "f"(0.f) : "memory");
}

// HALF (option "vl_half", a measurement of Newton's third law on this path): the lists hold
// every pair once; the force on i is summed in registers and added to frc[i] at the end, the reaction goes to
// frc[j] pair by pair through red.global.add.v4.f32; frc is zeroed before the launch.
// Fused integrator of the list path (option "vl_fuse"): what the epilogue of k_vl_force<.., FUSED> needs.
struct VlFuse {
    float4 *pos, *vel, *lnext;        // lnext: the local coordinates of the next step (the others read lpos meanwhile)
    const float4 *lbuild;
    VlCtl *ctl;
    float hdt, dt;
};

// FUSED (full lists only): the thread that owns F_i applies the closing half-kick of this step and the opening
// half-kick, drift, wrap, local coordinate and displacement check of the next one (the arithmetic of
// k_vl_kick_drift<2>): slots are stable between rebuilds, so an interior step is this one kernel plus the
// conditional build launches.
template <bool MODE2, bool HALF, bool FUSED>
__global__ void __launch_bounds__(VL_T, VL_MINB)
k_vl_force(const float4 *__restrict__ lpos, int N, int npad, Grid g, PairParams P, VlConst K,
           const unsigned *__restrict__ list, const int *__restrict__ count, float4 *__restrict__ frc,
           double *__restrict__ part_pe, double *__restrict__ part_w, VlFuse U)
{
    __shared__ float4 offt[128];
    __shared__ unsigned queue[VL_Q][VL_T];
    __shared__ double red[32];
    for (int t = threadIdx.x; t < 125; t += VL_T)
        offt[t] = make_float4(vl_code_value(t % 5, g), vl_code_value((t / 5) % 5, g), vl_code_value(t / 25, g), 0.f);
    __syncthreads();
    const int i = blockIdx.x * VL_T + threadIdx.x;
    double pe = 0.0, w = 0.0;
    float d2move = 0.f;
    if (i < N) {
        const float4 li = lpos[i];
        const int cnt = count[i];
        float fx = 0.f, fy = 0.f, fz = 0.f, sA = 0.f, sB = 0.f, sR = 0.f;
        int nin = 0, nq = 0;
        const unsigned *row = list + i;
        // four list entries per iteration: the coalesced list reads and the four gathers are all
        // issued before the first pair term (the kernel is bound by the latency of the gathers)
        // (the builders pad every list to a multiple of VL_U entries with inert ones: no validity tests here)
        const size_t stride = (size_t)npad;
        for (int k = 0; k < cnt; k += VL_U, row += VL_U * stride) {
            unsigned e[VL_U];
            float4 lj[VL_U];
#pragma unroll
            for (int u = 0; u < VL_U; u++) e[u] = row[u * stride];
#pragma unroll
            for (int u = 0; u < VL_U; u++) lj[u] = lpos[e[u] & VL_JMASK];
#pragma unroll
            for (int u = 0; u < VL_U; u++) {
                const float4 o = offt[e[u] >> 23];
                const float dx = (lj[u].x - li.x) + o.x, dy = (lj[u].y - li.y) + o.y, dz = (lj[u].z - li.z) + o.z;
                const float r2 = fmaf(dx, dx, fmaf(dy, dy, dz * dz));
                // p2 <= r2 < rc2_lo: FP32 term; the steep part and the sliver around rc^2: FP64 (queued)
                const bool fast = r2 >= K.p2 && r2 < K.rc2_lo;
                if (!fast && r2 < K.rc2_hi) {
                    queue[min(nq, VL_Q - 1)][threadIdx.x] = e[u];
                    nq++;
                }
                float inv;
                asm("rcp.approx.ftz.f32 %0, %1;" : "=f"(inv) : "f"(r2));
                inv = fmaf(inv, fmaf(-r2, inv, 1.f), inv);
                const float s2 = K.sig2 * inv;
                float s6 = s2 * s2 * s2;
                s6 = fast ? s6 : 0.f;
                float fr = inv * s6 * fmaf(K.eps48, s6, -K.eps24);
                if (MODE2) {
                    const float r = sqrtf(r2);
                    fr -= fast ? P.f_rcf * inv * r : 0.f;
                    sR += fast ? (r - P.rcf) : 0.f;
                }
                fx = fmaf(-fr, dx, fx);
                fy = fmaf(-fr, dy, fy);
                fz = fmaf(-fr, dz, fz);
                if (HALF && fast) vl_react(frc, (int)(e[u] & VL_JMASK), fr * dx, fr * dy, fr * dz);
                sA = fmaf(s6, s6, sA);
                sB += s6;
                nin += fast ? 1 : 0;
            }
        }
        // FP64 part: the queued pairs; a thread whose queue overflowed rescans its list instead
        double dfx = 0.0, dfy = 0.0, dfz = 0.0, dpe = 0.0, dw = 0.0;
        if (nq <= VL_Q) {
            for (int q = 0; q < nq; q++) {
                const unsigned e = queue[q][threadIdx.x];
                double px = 0.0, py = 0.0, pz = 0.0;
                vl_precise(lpos, offt, P, li, e, px, py, pz, dpe, dw);
                dfx += px; dfy += py; dfz += pz;
                if (HALF) vl_react(frc, (int)(e & VL_JMASK), (float)-px, (float)-py, (float)-pz);
            }
        } else {
            row = list + i;
            for (int k = 0; k < cnt; k++) {
                const unsigned e = row[(size_t)k * npad];
                const float4 lj = lpos[e & VL_JMASK];
                const float4 o = offt[e >> 23];
                const float dx = (lj.x - li.x) + o.x, dy = (lj.y - li.y) + o.y, dz = (lj.z - li.z) + o.z;
                const float r2 = fmaf(dx, dx, fmaf(dy, dy, dz * dz));
                if (!(r2 >= K.p2 && r2 < K.rc2_lo) && r2 < K.rc2_hi) {
                    double px = 0.0, py = 0.0, pz = 0.0;
                    vl_precise(lpos, offt, P, li, e, px, py, pz, dpe, dw);
                    dfx += px; dfy += py; dfz += pz;
                    if (HALF) vl_react(frc, (int)(e & VL_JMASK), (float)-px, (float)-py, (float)-pz);
                }
            }
        }
        const float Fx = (float)(dfx + (double)fx), Fy = (float)(dfy + (double)fy), Fz = (float)(dfz + (double)fz);
        if (HALF) vl_react(frc, i, Fx, Fy, Fz);
        else if (!FUSED) frc[i] = make_float4(Fx, Fy, Fz, 0.f);
        else {
            float4 p = U.pos[i], v = U.vel[i];
#pragma unroll
            for (int k = 0; k < 2; k++) {
                v.x = fmaf(U.hdt, Fx, v.x);
                v.y = fmaf(U.hdt, Fy, v.y);
                v.z = fmaf(U.hdt, Fz, v.z);
            }
            p.x = wrap_drift(fmaf(U.dt, v.x, p.x), g.L);
            p.y = wrap_drift(fmaf(U.dt, v.y, p.y), g.L);
            p.z = wrap_drift(fmaf(U.dt, v.z, p.z), g.L);
            const int c = __float_as_int(li.w) & VL_CELLMASK;
            const int cz = c % g.n, cy = (c / g.n) % g.n, cx = c / (g.n * g.n);
            float4 l;
            l.x = vl_local(p.x, cx, g);
            l.y = vl_local(p.y, cy, g);
            l.z = vl_local(p.z, cz, g);
            l.w = li.w;
            U.pos[i] = p;
            U.vel[i] = v;
            U.lnext[i] = l;
            const float4 l0 = U.lbuild[i];
            const float ex = l.x - l0.x, ey = l.y - l0.y, ez = l.z - l0.z;
            d2move = fmaf(ex, ex, fmaf(ey, ey, ez * ez));
        }
        pe = dpe + P.eps4 * ((double)sA - (double)sB) - (double)nin * P.ushift;
        w = dw + P.eps24 * (2.0 * (double)sA - (double)sB);
        if (MODE2) {
            pe += P.f_rc * (double)sR;
            w -= P.f_rc * ((double)sR + (double)nin * P.rc);
        }
    }
    if (FUSED) {
        d2move = fmaxf(d2move, __shfl_xor_sync(0xffffffffu, d2move, 16));
        d2move = fmaxf(d2move, __shfl_xor_sync(0xffffffffu, d2move, 8));
        d2move = fmaxf(d2move, __shfl_xor_sync(0xffffffffu, d2move, 4));
        d2move = fmaxf(d2move, __shfl_xor_sync(0xffffffffu, d2move, 2));
        d2move = fmaxf(d2move, __shfl_xor_sync(0xffffffffu, d2move, 1));
        if ((threadIdx.x & 31) == 0 && d2move > 0.f) atomicMax(&U.ctl->maxd2, __float_as_uint(d2move));
    }
    pe = block_sum(pe, red);
    w = block_sum(w, red);
    if (threadIdx.x == 0) {
        part_pe[blockIdx.x] = (HALF ? 1.0 : 0.5) * pe;              // full lists: every pair is in both atoms' lists
        part_w[blockIdx.x] = (HALF ? 1.0 : 0.5) * w;
    }
}

// ---------------------------------------------------------------------------------------
// Host side.
// Control block and build-time coordinates: shared by the neighbour-list path and the skin-cell path.
static int vl_alloc_base(md_sim *s)
{
    if (s->vl_ctl) return MD_OK;
    s->vl_lbuild = (float4 *)ljmd_dev_alloc((size_t)s->N * sizeof(float4), s->stream);
    s->vl_ctl = (VlCtl *)ljmd_dev_alloc(sizeof(VlCtl), s->stream);
    s->lpos2 = (float4 *)ljmd_dev_alloc((size_t)s->N * sizeof(float4), s->stream);
    if (!s->vl_lbuild || !s->vl_ctl || !s->lpos2) {
        ljmd_dev_free(s->vl_lbuild, s->stream); ljmd_dev_free(s->vl_ctl, s->stream); ljmd_dev_free(s->lpos2, s->stream);
        s->vl_lbuild = nullptr; s->vl_ctl = nullptr; s->lpos2 = nullptr;
        return MD_ENOMEM;
    }
    CK(cudaMemsetAsync(s->vl_ctl, 0, sizeof(VlCtl), s->stream));
    return MD_OK;
}

static int vl_alloc(md_sim *s)
{
    if (s->vl_list) return MD_OK;
    int r0 = vl_alloc_base(s);
    if (r0) return r0;
    const Grid &g = s->vgrid;
    if (s->N > (int64_t)VL_JMASK) return MD_EUNSUPPORTED;               // slot index must fit 23 bits
    const double rl = s->rc + s->skin;
    const double mean = 4.0 / 3.0 * 3.14159265358979 * rl * rl * rl * (double)s->N / (s->L * s->L * s->L);
    int cap = (int)(1.4 * mean) + 32;
    cap = (cap + 7) / 8 * 8;                                            // a multiple of VL_U: padding always fits
    s->vl_cap = cap;
    s->vl_npad = (int)((s->N + 31) / 32 * 32);
    s->vl_list = (unsigned *)ljmd_dev_alloc((size_t)cap * s->vl_npad * sizeof(unsigned), s->stream);
    s->vl_count = (int *)ljmd_dev_alloc((size_t)s->N * sizeof(int), s->stream);
    if (!s->vl_list || !s->vl_count) {
        ljmd_dev_free(s->vl_list, s->stream); ljmd_dev_free(s->vl_count, s->stream);
        s->vl_list = nullptr; s->vl_count = nullptr;
        return MD_ENOMEM;
    }
    (void)g;
    return MD_OK;
}

// After an overflow: lists long enough for `need` entries (plus a margin); the next evaluation rebuilds.
int ljmd_vl_grow(md_sim *s, int need)
{
    int cap = need + need / 8 + 8;
    cap = (cap + 7) / 8 * 8;
    if (cap <= s->vl_cap) return MD_OK;
    CK(cudaStreamSynchronize(s->stream));
    unsigned *nl = (unsigned *)ljmd_dev_alloc((size_t)cap * s->vl_npad * sizeof(unsigned), s->stream);
    if (!nl) return MD_ENOMEM;
    ljmd_dev_free(s->vl_list, s->stream);
    s->vl_list = nl;
    s->vl_cap = cap;
    ljmd_drop_graphs(s);                                 // captured build and force kernels hold the old pointer and capacity
    s->layout = LAYOUT_NONE;                             // forces a build at the next evaluation
    return MD_OK;
}

// Ask for a build at the next force evaluation (state set from outside, other path used in between).
static int vl_force_build(md_sim *s)
{
    const int one = 1;
    CK(cudaMemcpyAsync(&s->vl_ctl->force, &one, sizeof(int), cudaMemcpyHostToDevice, s->stream));
    CK(cudaStreamSynchronize(s->stream));                                // `one` is on the stack
    return MD_OK;
}

int ljmd_vl_kick_drift(md_sim *s, int kicks)
{
    const int N = (int)s->N, nb = (N + 255) / 256;
    if (kicks == 2)
        k_vl_kick_drift<2><<<nb, 256, 0, s->stream>>>(s->pos, s->vel, s->frc, s->lpos, s->vl_lbuild, N, s->hdtf, s->dtf,
                                                      s->vgrid, s->vl_ctl);
    else
        k_vl_kick_drift<1><<<nb, 256, 0, s->stream>>>(s->pos, s->vel, s->frc, s->lpos, s->vl_lbuild, N, s->hdtf, s->dtf,
                                                      s->vgrid, s->vl_ctl);
    CKL(s);
    return MD_OK;
}

// Decide on the device whether the skin has been used up, and if so re-sort the atoms into the cells of
// s->vgrid (histogram, scan, scatter, copy back: every kernel returns at once when the flag is clear).
static int vl_decide_and_sort(md_sim *s, int layout)
{
    int r;
    const int N = (int)s->N;
    const int nb = min((N + 255) / 256, 148 * 16);            // grid-stride kernels: idle launches stay cheap
    const Grid &g = s->vgrid;
    if (s->layout != layout) {
        if ((r = vl_force_build(s))) return r;
        s->layout = layout;
    }
    const float half = 0.5f * (float)s->skin;
    float thr = half * half;
    unsigned thr_bits;
    memcpy(&thr_bits, &thr, sizeof(thr_bits));
    k_vl_decide<<<1, 1, 0, s->stream>>>(s->vl_ctl, thr_bits);
    CKL(s);
    k_vl_bin<<<nb, 256, 0, s->stream>>>(s->pos, N, g, s->cell_of, s->rank, s->cell_count, s->vl_ctl);
    CKL(s);
    if ((r = ljmd_scan_counts(s, s->cell_count, s->cell_start, g.ncells, &s->vl_ctl->rebuild))) return r;
    k_vl_scatter<<<nb, 256, 0, s->stream>>>(s->pos, s->vel, N, g, s->cell_of, s->rank, s->cell_start, s->pos2, s->vel2,
                                            s->lpos, s->vl_ctl);
    CKL(s);
    k_vl_copyback<<<nb, 256, 0, s->stream>>>(s->pos, s->vel, s->vl_lbuild, s->pos2, s->vel2, s->lpos, N, s->vl_ctl);
    CKL(s);
    return MD_OK;
}

// Skin cells ("use an even larger skin and therefore update the cell lists
// only every couple of time steps"): cells of side >= rc + skin; between rebuilds every atom keeps its slot
// and home cell, the integrator keeps its local coordinate in that cell's frame (k_vl_kick_drift), and the
// cell-force kernel runs on those cells with the exact cutoff rc.  An atom strays at most skin / 2 from where
// it was at the last rebuild before the device-side decision re-sorts, so no pair inside rc is ever outside the
// 27 home cells.  Same forces as the rebuild-every-step path.
int ljmd_forces_skincell(md_sim *s, bool energy)
{
    int r = vl_alloc_base(s);
    if (r) return r;
    if ((r = vl_decide_and_sort(s, LAYOUT_SKINCELL))) return r;
    ljmd_tick(s, TAG_BUILD);
    return ljmd_forces_cell2_on(s, s->vgrid, 0.5 * s->skin, energy, false);
}

// Decide, (re)build if the device-side flag says so, evaluate forces from the lists.
int ljmd_forces_verlet(md_sim *s, bool fuse)
{
    int r = vl_alloc(s);
    if (r) return r;
    s->fused_pending = false;
    fuse = fuse && !s->vl_half;
    const int N = (int)s->N, nbl = (N + VL_T - 1) / VL_T;
    const Grid &g = s->vgrid;
    if ((r = vl_decide_and_sort(s, LAYOUT_VERLET))) return r;
    const double rl = s->rc + s->skin;
    if (s->vl_naive_build || s->vl_half) {
        k_vl_build<<<nbl, VL_T, 0, s->stream>>>(s->lpos, s->cell_start, N, s->vl_npad, g, (float)(rl * rl), s->vl_cap, s->vl_list,
                                                s->vl_count, s->vl_ctl, s->vl_half ? 1 : 0);
        CKL(s);
    } else if ((r = ljmd_vl_build_lists(s, &s->vl_ctl->rebuild))) return r;
    ljmd_tick(s, TAG_BUILD);
    if (nbl > s->part_cap) return MD_ENOMEM;
    double *ppe = s->part + (size_t)s->part_cap;
    double *pw = s->part + 2 * (size_t)s->part_cap;
    const PairParams &P = s->pp;
    VlConst K;
    K.rc2_lo = (float)(P.rc2 * (1.0 - 4e-6));
    K.rc2_hi = (float)(P.rc2 * (1.0 + 4e-6));
    K.p2 = (float)fmin(P.precise_r2, 3.0e38);
    K.sig2 = P.sig2f;
    K.eps24 = P.eps24f;
    K.eps48 = 2.0f * P.eps24f;
    {
        // the kernel is bound by its gathers: leave the unified L1 / shared memory mostly to the L1
        // (30 % still holds eight blocks' tables and queues); measured 3 % faster than the default split
        static bool carved = false;
        if (!carved) {
            cudaFuncSetAttribute(k_vl_force<false, false, false>, cudaFuncAttributePreferredSharedMemoryCarveout, 30);
            cudaFuncSetAttribute(k_vl_force<true, false, false>, cudaFuncAttributePreferredSharedMemoryCarveout, 30);
            cudaFuncSetAttribute(k_vl_force<false, true, false>, cudaFuncAttributePreferredSharedMemoryCarveout, 30);
            cudaFuncSetAttribute(k_vl_force<true, true, false>, cudaFuncAttributePreferredSharedMemoryCarveout, 30);
            cudaFuncSetAttribute(k_vl_force<false, false, true>, cudaFuncAttributePreferredSharedMemoryCarveout, 30);
            cudaFuncSetAttribute(k_vl_force<true, false, true>, cudaFuncAttributePreferredSharedMemoryCarveout, 30);
            carved = true;
        }
    }
    if (s->vl_half) CK(cudaMemsetAsync(s->frc, 0, (size_t)N * sizeof(float4), s->stream));
    VlFuse U;
    U.pos = s->pos; U.vel = s->vel; U.lnext = s->lpos2; U.lbuild = s->vl_lbuild; U.ctl = s->vl_ctl;
    U.hdt = s->hdtf; U.dt = s->dtf;
#define VL_LAUNCH(M2, H, F) \
    k_vl_force<M2, H, F><<<nbl, VL_T, 0, s->stream>>>(s->lpos, N, s->vl_npad, g, P, K, s->vl_list, s->vl_count, s->frc, ppe, pw, U)
    if (fuse) { if (P.mode == 2) VL_LAUNCH(true, false, true); else VL_LAUNCH(false, false, true); }
    else if (P.mode == 2) { if (s->vl_half) VL_LAUNCH(true, true, false); else VL_LAUNCH(true, false, false); }
    else { if (s->vl_half) VL_LAUNCH(false, true, false); else VL_LAUNCH(false, false, false); }
#undef VL_LAUNCH
    if (fuse) {                                          // the next step reads what this epilogue wrote
        float4 *t = s->lpos; s->lpos = s->lpos2; s->lpos2 = t;
        s->fused_pending = true;
    }
    CKL(s);
    ljmd_tick(s, TAG_FORCE);
    s->n_pe = nbl;
    return MD_OK;
}

// List statistics for md_get_stat: builds and steps so far, overflow flag.
int ljmd_vl_stats(md_sim *s, int *nbuilds, int *nsteps, int *overflow)
{
    *nbuilds = *nsteps = *overflow = 0;
    if (!s->vl_ctl) return MD_OK;
    VlCtl h;
    CK(cudaMemcpyAsync(&h, s->vl_ctl, sizeof(h), cudaMemcpyDeviceToHost, s->stream));
    CK(cudaStreamSynchronize(s->stream));
    *nbuilds = h.nbuilds;
    *nsteps = h.nsteps;
    *overflow = h.overflow;
    return MD_OK;
}
