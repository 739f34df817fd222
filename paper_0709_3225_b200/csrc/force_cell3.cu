// Cell-list Lennard-Jones force, third generation: dense evaluation (in its
// fused form, a1/a5; one block per cell, every atom of the 27 neighbour cells staged
// through shared memory and the force evaluated for every staged pair, no neighbour bookkeeping).
//
// The first two kernels (force_cell.cu, force_cell2.cu) filter the 27 x occupancy candidates with a
// ballot and walk the hit bits per lane; ncu showed them issuing mostly integer and shared-memory
// bookkeeping (FMA pipe 35 % busy, 31 warp instructions per hit at 53 % lane utilisation).  Here the
// paper's own structure is taken back: every staged candidate is evaluated, with nothing to keep
// track of, and the arithmetic is packed two candidates per instruction (FADD2/FMUL2/FFMA2).
// MEASURED SLOWER than the ballot kernel (0.138 against 0.101 ms per force launch at N = 256,000; DESIGN.md
// section 7): a packed instruction holds the issue port for two cycles on B200, so the loop costs 110 cycles per
// four candidates, 27.5 issue slots per (atom, candidate), and 263 candidates per atom lose against filtering 351
// and evaluating 52.  Kept as option "cell_kernel" = 3 and as an independent cross-check.  What keeps it cheap:
//   * candidates farther than rc from the home cell's box are dropped while staging (a ball-inflated
//     box holds 20.6 cell volumes instead of 27), compacted with one ballot per 32 candidates;
//   * lane = (atom i of the cell, slice of the candidate quads), floor(32 / atoms) slices per atom, one
//     LDS.128 per coordinate and four candidates, all lanes the same trip count, no branches;
//   * FP32 terms only inside the window p2 <= r^2 < rc^2 (1 - 4e-6) (one FADD2 + compare on |r^2 - mid|);
//     everything else that may be inside rc (the steep part, the sliver around rc^2, the atom itself) is
//     pushed on a per-lane queue and evaluated in FP64 from the exact coordinates;
//   * FUSED: the lane that owns F_i applies the closing half-kick of this step and the opening half-kick,
//     drift, wrap and cell histogram of the next one (same FMAs as k_kick_drift_bin<2>), so an interior
//     step of md_step is force kernel + scan + scatter and the forces never travel through HBM.
// Positions are read as stored (global coordinates); the exact cell-local frame of DESIGN.md section 5
// is rebuilt per candidate as (x - origin of its cell) + (offset between the two cells - h).
#include <math.h>
#include "common.cuh"
#include "pair.cuh"

#define F3_CAP 416                    // compacted candidates per staging pass (27 cells of 13 atoms keep ~265)
#define F3_TILE (F3_CAP + 64)         // plus one more row of 27 and the padding to a multiple of 4 x slices
#define F3_QCAP 10                    // queued FP64 pairs per lane (row F3_QCAP is the overflow sentinel)
#ifndef F3_MINB
#define F3_MINB 28                    // resident one-warp blocks per SM
#endif
#define F3_FULL 0xffffffffu
#define F3_NSEG 27

struct F3Smem {
    float t[3][F3_TILE];              // compacted candidates, u = position in the home cell's centred frame
    unsigned short raw[F3_TILE];      // (neighbour cell) | (atom of that cell - first atom of the pass) << 5
    unsigned short q[F3_QCAP + 1][32];
};

struct F3Const {
    float mid, hw, hw2;               // FP32 window |r2 - mid| < hw; FP64 queue when outside it and r2 - mid < hw2
    float p2, rc2_lo;                 // the same window as bounds (overflow rescan)
    float prune2;                     // squared reach of the home box
    float sig2, eps24, neps48;
    float h;                          // half a cell side: centre of the frame
    float f_rcf, rcf;                 // mode 2
    float hdt, dt;                    // fused integrator
    double hd;
    int tile_exact;                   // staged FP32 coordinates are exact away from the box origin
};

__device__ __forceinline__ float f3_rcp(float x)
{
    float y;
    asm("rcp.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x));
    return y;
}

// Append candidate number `c` to the lane's FP64 queue when `push`; the write pointer stops at qend.
__device__ __forceinline__ void f3_push(unsigned &qa, int c, bool push, unsigned qend)
{
    asm volatile("{ .reg .pred p;\n\t setp.ne.b32 p, %2, 0;\n\t @p st.shared.u16 [%0], %1;\n\t }"
                 :: "r"(qa), "h"((unsigned short)c), "r"((int)push) : "memory");
    qa = push ? min(qa + 64u, qend) : qa;
}

// FP64 pair term without branches: a pair with r^2 >= rc^2, the atom itself (r^2 = 0) or an idle slot
// (far-away displacement) contributes exactly zero.
template <bool MODE2, bool ENERGY>
__device__ __forceinline__ void f3_pair64(const PairParams &P, double dx, double dy, double dz, double &fx,
                                          double &fy, double &fz, double &pe, double &w)
{
    const double r2 = fma(dx, dx, fma(dy, dy, dz * dz));
    const bool in = r2 < P.rc2 && r2 > 0.0;              // strict
    if (P.kind == 1) {                                   // Yukawa (pair.cuh): rare path, a branch is fine
        if (in && r2 > 0.0) {
            double fr_, u_;
            yukawa_fu64(P, r2, fr_, u_);
            fx = fma(-fr_, dx, fx);
            fy = fma(-fr_, dy, fy);
            fz = fma(-fr_, dz, fz);
            if (ENERGY) {
                pe += u_;
                w = fma(fr_, r2, w);
            }
        }
        return;
    }
    const double inv = in ? rcp_f64(r2) : 0.0;
    const double s2 = P.sig2 * inv;
    const double s6 = s2 * s2 * s2;
    double fr = P.eps24 * inv * s6 * (2.0 * s6 - 1.0);
    double u = in ? P.eps4 * s6 * (s6 - 1.0) - P.ushift : 0.0;
    if (MODE2) {                                         // PAPER.md:61 (Eq. 3): f = f_LJ(r) - f_LJ(rc)
        const double r = sqrt(r2);
        u += in ? (r - P.rc) * P.f_rc : 0.0;
        fr -= P.f_rc * inv * r;
    }
    fx = fma(-fr, dx, fx);
    fy = fma(-fr, dy, fy);
    fz = fma(-fr, dz, fz);
    if (ENERGY) {
        pe += u;
        w = fma(fr, in ? r2 : 0.0, w);
    }
}

struct F3Acc {
    float2 fx, fy, fz, sA, sB, cnt;
    float sR;
};

// Two candidates (c, c + 1) against the lane's atom, packed.  nU = -u_i.
template <bool MODE2, bool ENERGY>
__device__ __forceinline__ void f3_pair2(const float2 X, const float2 Y, const float2 Z, const float2 nUX,
                                         const float2 nUY, const float2 nUZ, const F3Const &K, F3Acc &A,
                                         unsigned &qa, const unsigned qend, const int c)
{
    const float2 dx = __fadd2_rn(X, nUX), dy = __fadd2_rn(Y, nUY), dz = __fadd2_rn(Z, nUZ);
    const float2 r2 = __ffma2_rn(dx, dx, __ffma2_rn(dy, dy, __fmul2_rn(dz, dz)));
    const float2 t = __fadd2_rn(r2, make_float2(-K.mid, -K.mid));
    const bool in0 = fabsf(t.x) < K.hw, in1 = fabsf(t.y) < K.hw;
    f3_push(qa, c, !in0 && t.x < K.hw2, qend);
    f3_push(qa, c + 1, !in1 && t.y < K.hw2, qend);
    float2 inv = make_float2(f3_rcp(r2.x), f3_rcp(r2.y));
    inv = __ffma2_rn(inv, __ffma2_rn(make_float2(-r2.x, -r2.y), inv, make_float2(1.f, 1.f)), inv);   // one Newton step
    // outside the FP32 window the pair contributes nothing here: 1/r^2 := 0 (also swallows the inf/NaN of
    // the atom itself)
    inv.x = in0 ? inv.x : 0.f;
    inv.y = in1 ? inv.y : 0.f;
    const float2 s2 = __fmul2_rn(make_float2(K.sig2, K.sig2), inv);
    const float2 s6 = __fmul2_rn(__fmul2_rn(s2, s2), s2);
    // -f/r = inv s6 (24 eps - 48 eps s6)
    float2 nfr = __fmul2_rn(__fmul2_rn(inv, s6), __ffma2_rn(make_float2(K.neps48, K.neps48), s6, make_float2(K.eps24, K.eps24)));
    if (MODE2) {
        const float r0 = sqrtf(r2.x), r1 = sqrtf(r2.y);
        nfr.x += in0 ? K.f_rcf * inv.x * r0 : 0.f;
        nfr.y += in1 ? K.f_rcf * inv.y * r1 : 0.f;
        if (ENERGY) {
            A.sR += in0 ? (r0 - K.rcf) : 0.f;
            A.sR += in1 ? (r1 - K.rcf) : 0.f;
        }
    }
    A.fx = __ffma2_rn(nfr, dx, A.fx);
    A.fy = __ffma2_rn(nfr, dy, A.fy);
    A.fz = __ffma2_rn(nfr, dz, A.fz);
    if (ENERGY) {
        A.sA = __ffma2_rn(s6, s6, A.sA);
        A.sB = __fadd2_rn(A.sB, s6);
        A.cnt = __fadd2_rn(A.cnt, make_float2(in0 ? 1.f : 0.f, in1 ? 1.f : 0.f));
    }
}

template <bool MODE2, bool ENERGY, bool FUSED>
__global__ void __launch_bounds__(32, F3_MINB)
k_fc3(const float4 *__restrict__ pos, const int *__restrict__ cell_start, const Grid g, const PairParams P,
      const F3Const K, float4 *__restrict__ frc, double *__restrict__ part_pe, double *__restrict__ part_w,
      const int nmax, float4 *__restrict__ vel, float4 *__restrict__ pos_out, int *__restrict__ cell_count)
{
    __shared__ __align__(16) F3Smem S;
    const int lane = threadIdx.x;
    const int n = g.n;
    int cz = blockIdx.x, cy = blockIdx.y, cx = blockIdx.z;
    if (g.morton) {                                      // 1-D grid over the padded cube, blocks in Morton order
        cz = (int)morton_compact(blockIdx.x);
        cy = (int)morton_compact(blockIdx.x >> 1);
        cx = (int)morton_compact(blockIdx.x >> 2);
        if (cx >= n || cy >= n || cz >= n) return;
    }
    const int home = cell_id(cx, cy, cz, g);
    double pe_tot = 0.0, w_tot = 0.0;
    // ---- the 27 neighbour cells ("segments"): first slot, count, origin, exact origin offset
    int cnt = 0, start = 0;
    float ox = 0.f, oy = 0.f, oz = 0.f, ax_o = 0.f, ay_o = 0.f, az_o = 0.f;
    if (lane < F3_NSEG) {
        const int col = lane / 3, dz = lane - col * 3 - 1;
        const int ax = col / 3 - 1, ay = col - (col / 3) * 3 - 1;
        int nx = cx + ax, ny = cy + ay, nz = cz + dz;
        nx += (nx < 0) ? n : 0; nx -= (nx >= n) ? n : 0;
        ny += (ny < 0) ? n : 0; ny -= (ny >= n) ? n : 0;
        nz += (nz < 0) ? n : 0; nz -= (nz >= n) ? n : 0;
        // distance between the cell origins: exact
        ox = (ax == 0) ? 0.f : (ax > 0 ? ((cx == n - 1) ? g.last : g.side) : -((nx == n - 1) ? g.last : g.side));
        oy = (ay == 0) ? 0.f : (ay > 0 ? ((cy == n - 1) ? g.last : g.side) : -((ny == n - 1) ? g.last : g.side));
        oz = (dz == 0) ? 0.f : (dz > 0 ? ((cz == n - 1) ? g.last : g.side) : -((nz == n - 1) ? g.last : g.side));
        ax_o = (float)nx * g.side; ay_o = (float)ny * g.side; az_o = (float)nz * g.side;
        const int nb = cell_id(nx, ny, nz, g);
        start = cell_start[nb];
        cnt = cell_start[nb + 1] - start;
    }
    const int ibeg = cell_start[home], ni = cell_start[home + 1] - ibeg;
    if (ni > 0) {
        const int maxcnt = __reduce_max_sync(F3_FULL, cnt);
        // the home cell's box in the centred frame: [-h, width - h] per dimension
        const float bx = ((cx == n - 1) ? g.last : g.side) - K.h, by = ((cy == n - 1) ? g.last : g.side) - K.h,
                    bz = ((cz == n - 1) ? g.last : g.side) - K.h;
        const float hox = (float)cx * g.side, hoy = (float)cy * g.side, hoz = (float)cz * g.side;
        // no staged cell has index 0 in any dimension: every global coordinate is >= side >= 2
        const bool exact = K.tile_exact && cx >= 2 && cx <= n - 2 && cy >= 2 && cy <= n - 2 && cz >= 2 && cz <= n - 2;
        const float sbx = ox - K.h, sby = oy - K.h, sbz = oz - K.h;
        const unsigned lt = (1u << lane) - 1u;
        int staged_kbeg = -1, staged_kend = 0, m = 0;

        for (int i0 = 0; i0 < ni; i0 += 32) {
            // ---- lanes of this pass: nrow atoms, SL slices of the candidate quads per atom
            const int nrow = min(32, ni - i0);
            int SL = 32 / nrow;
            SL = (SL > 4) ? ((SL >= 8) ? 8 : 4) : SL;
            const float invrow = __frcp_rn((float)nrow);
            const int sl = (int)(((float)lane + 0.5f) * invrow), li_ = lane - sl * nrow;
            const bool myvalid = sl < SL;
            const int myslot = ibeg + i0 + (myvalid ? li_ : 0);
            const float4 pme = pos[myslot];
            float4 vme;
            if (FUSED) vme = vel[myslot];                        // early: its latency hides behind the whole pass
            const float ux = (pme.x - hox) - K.h, uy = (pme.y - hoy) - K.h, uz = (pme.z - hoz) - K.h;
            const float2 nUX = make_float2(-ux, -ux), nUY = make_float2(-uy, -uy), nUZ = make_float2(-uz, -uz);
            F3Acc A;
            A.fx = A.fy = A.fz = A.sA = A.sB = A.cnt = make_float2(0.f, 0.f);
            A.sR = 0.f;
            double dfx = 0.0, dfy = 0.0, dfz = 0.0, dpe = 0.0, dw = 0.0;

            for (int kbeg = 0; kbeg < maxcnt; kbeg = staged_kend) {
                if (kbeg != staged_kbeg) {
                    // ---- stage atoms kbeg, kbeg + 1, ... of every neighbour cell (lane = cell), keeping those
                    // within rc of the home box, until the tile is full
                    staged_kbeg = kbeg;
                    __syncwarp();
                    m = 0;
                    int k = kbeg;
                    const int klim = min(maxcnt, kbeg + 1024);
                    for (; k < klim && m <= F3_CAP - 108; k += 4) {
                        float4 p[4];
#pragma unroll
                        for (int u = 0; u < 4; u++) p[u] = pos[min(max(start + k + u, 0), nmax)];
#pragma unroll
                        for (int u = 0; u < 4; u++) {
                            const float x = (p[u].x - ax_o) + sbx;
                            const float y = (p[u].y - ay_o) + sby;
                            const float z = (p[u].z - az_o) + sbz;
                            const float ex = fmaxf(fmaxf(-K.h - x, x - bx), 0.f);
                            const float ey = fmaxf(fmaxf(-K.h - y, y - by), 0.f);
                            const float ez = fmaxf(fmaxf(-K.h - z, z - bz), 0.f);
                            const bool keep = k + u < cnt && fmaf(ex, ex, fmaf(ey, ey, ez * ez)) < K.prune2;
                            const unsigned bal = __ballot_sync(F3_FULL, keep);
                            if (keep) {
                                const int d = m + __popc(bal & lt);
                                S.t[0][d] = x;
                                S.t[1][d] = y;
                                S.t[2][d] = z;
                                S.raw[d] = (unsigned short)(lane | ((k + u - kbeg) << 5));
                            }
                            m += __popc(bal);
                        }
                    }
                    staged_kend = min(k, maxcnt);
                    // far-away entries up to the next multiple of four plus seven quads (the trip count is
                    // rounded up to a multiple of the slice count, at most 8)
                    for (int d = m + lane; d < ((m + 3) & ~3) + 60; d += 32) {
                        S.t[0][d] = 1.0e4f;
                        S.t[1][d] = 1.0e4f;
                        S.t[2][d] = 1.0e4f;
                        S.raw[d] = 0;
                    }
                }
                __syncwarp();
                // ---- dense loop over my quads q = sl, sl + SL, ...
                const int nq = (((m + 3) >> 2) + 2 * SL - 1) / (2 * SL) * (2 * SL);    // same, even trip count for every slice
                const unsigned q0 = (unsigned)__cvta_generic_to_shared(&S.q[0][lane]);
                unsigned qa = q0;
                const unsigned qend = q0 + F3_QCAP * 64u;
                const float4 *tx4 = reinterpret_cast<const float4 *>(&S.t[0][0]);
                const float4 *ty4 = reinterpret_cast<const float4 *>(&S.t[1][0]);
                const float4 *tz4 = reinterpret_cast<const float4 *>(&S.t[2][0]);
#ifndef F3_SKIP_DENSE
                if (myvalid) {
                    for (int q = sl; q < nq; q += 2 * SL) {
                        const float4 X = tx4[q], Y = ty4[q], Z = tz4[q];
                        const float4 X2 = tx4[q + SL], Y2 = ty4[q + SL], Z2 = tz4[q + SL];
                        f3_pair2<MODE2, ENERGY>(make_float2(X.x, X.y), make_float2(Y.x, Y.y), make_float2(Z.x, Z.y),
                                                nUX, nUY, nUZ, K, A, qa, qend, 4 * q);
                        f3_pair2<MODE2, ENERGY>(make_float2(X.z, X.w), make_float2(Y.z, Y.w), make_float2(Z.z, Z.w),
                                                nUX, nUY, nUZ, K, A, qa, qend, 4 * q + 2);
                        f3_pair2<MODE2, ENERGY>(make_float2(X2.x, X2.y), make_float2(Y2.x, Y2.y), make_float2(Z2.x, Z2.y),
                                                nUX, nUY, nUZ, K, A, qa, qend, 4 * (q + SL));
                        f3_pair2<MODE2, ENERGY>(make_float2(X2.z, X2.w), make_float2(Y2.z, Y2.w), make_float2(Z2.z, Z2.w),
                                                nUX, nUY, nUZ, K, A, qa, qend, 4 * (q + SL) + 2);
                    }
                }
#endif
                // ---- FP64 part of this pass: queued pairs from the exact coordinates; a lane whose queue
                // overflowed rescans its quads and takes every pair outside the FP32 window
                {
                    const bool ovf = qa == qend;
                    const int nq64 = ovf ? 0 : (int)(qa - q0) >> 6;
                    // exact displacement of compacted candidate c from my atom.  Away from the box origin the
                    // staged FP32 coordinates are exact (multiples of 2^-22 below 4: DESIGN.md section 5) and
                    // their difference is the displacement; otherwise it is rebuilt from the stored positions,
                    // the two cell origins and the exact origin offset.
                    auto disp = [&](const int c, double &ex, double &ey, double &ez) {
                        if (exact) {
                            ex = (double)S.t[0][c] - (double)ux;
                            ey = (double)S.t[1][c] - (double)uy;
                            ez = (double)S.t[2][c] - (double)uz;
                        } else {
                            // rare (cells touching the box origin): the candidate's cell from its number
                            const int rw = S.raw[c], sg = rw & 31;
                            const int col = sg / 3, ddz = sg - col * 3 - 1, dax = col / 3 - 1, day = col - (col / 3) * 3 - 1;
                            int nx = cx + dax, ny = cy + day, nz = cz + ddz;
                            nx += (nx < 0) ? n : 0; nx -= (nx >= n) ? n : 0;
                            ny += (ny < 0) ? n : 0; ny -= (ny >= n) ? n : 0;
                            nz += (nz < 0) ? n : 0; nz -= (nz >= n) ? n : 0;
                            const float qx = (dax == 0) ? 0.f : (dax > 0 ? ((cx == n - 1) ? g.last : g.side) : -((nx == n - 1) ? g.last : g.side));
                            const float qy = (day == 0) ? 0.f : (day > 0 ? ((cy == n - 1) ? g.last : g.side) : -((ny == n - 1) ? g.last : g.side));
                            const float qz = (ddz == 0) ? 0.f : (ddz > 0 ? ((cz == n - 1) ? g.last : g.side) : -((nz == n - 1) ? g.last : g.side));
                            const float4 pj = pos[min(cell_start[cell_id(nx, ny, nz, g)] + kbeg + (rw >> 5), nmax)];
                            ex = (((double)pj.x - (double)((float)nx * g.side)) + (double)qx) - ((double)pme.x - (double)hox);
                            ey = (((double)pj.y - (double)((float)ny * g.side)) + (double)qy) - ((double)pme.y - (double)hoy);
                            ez = (((double)pj.z - (double)((float)nz * g.side)) + (double)qz) - ((double)pme.z - (double)hoz);
                        }
                    };
#ifdef F3_SKIP_FP64
                    const int maxq = 0;
#else
                    const int maxq = __reduce_max_sync(F3_FULL, nq64);
#endif
                    for (int k = 0; k < maxq; k += 2) {          // two independent chains per iteration
                        double ax_ = 1.0e4, ay_ = 1.0e4, az_ = 1.0e4, bx_ = 1.0e4, by_ = 1.0e4, bz_ = 1.0e4;
                        if (k < nq64) disp((int)S.q[k][lane], ax_, ay_, az_);
                        if (k + 1 < nq64) disp((int)S.q[k + 1][lane], bx_, by_, bz_);
                        f3_pair64<MODE2, ENERGY>(P, ax_, ay_, az_, dfx, dfy, dfz, dpe, dw);
                        f3_pair64<MODE2, ENERGY>(P, bx_, by_, bz_, dfx, dfy, dfz, dpe, dw);
                    }
                    if (__any_sync(F3_FULL, ovf)) {
                        if (ovf) {
                            for (int q = sl; q < nq; q += SL) {
                                for (int k = 0; k < 4; k++) {
                                    const int c = 4 * q + k;
                                    const float ddx = S.t[0][c] - ux, ddy = S.t[1][c] - uy, ddz = S.t[2][c] - uz;
                                    const float tt = fmaf(ddx, ddx, fmaf(ddy, ddy, ddz * ddz)) - K.mid;
                                    if (!(fabsf(tt) < K.hw) && tt < K.hw2) {
                                        double ex, ey, ez;
                                        disp(c, ex, ey, ez);
                                        f3_pair64<MODE2, ENERGY>(P, ex, ey, ez, dfx, dfy, dfz, dpe, dw);
                                    }
                                }
                            }
                        }
                    }
                }
            }
            // ---- totals of this lane, reduction over the slices of an atom
            double tx_ = dfx + (double)A.fx.x + (double)A.fx.y;
            double ty_ = dfy + (double)A.fy.x + (double)A.fy.y;
            double tz_ = dfz + (double)A.fz.x + (double)A.fz.y;
            if (!myvalid) tx_ = ty_ = tz_ = 0.0;
            double ox_ = 0.0, oy_ = 0.0, oz_ = 0.0;
            for (int k = 1; k < SL; k++) {
                const int src = lane + k * nrow;                   // < 32 for the lanes of slice 0
                ox_ += __shfl_sync(F3_FULL, tx_, src);
                oy_ += __shfl_sync(F3_FULL, ty_, src);
                oz_ += __shfl_sync(F3_FULL, tz_, src);
            }
            if (sl == 0) {
                const float fx = (float)(tx_ + ox_), fy = (float)(ty_ + oy_), fz = (float)(tz_ + oz_);
                if (!FUSED) {
                    frc[myslot] = make_float4(fx, fy, fz, 0.f);
                } else {
                    // closing half-kick of this step, then the next step's half-kick, drift, wrap and cell
                    // histogram: the arithmetic of k_kick_drift_bin<2> (cells.cu) on the float force
                    float4 v = vme;
                    float4 p = pme;
#pragma unroll
                    for (int k = 0; k < 2; k++) {
                        v.x = fmaf(K.hdt, fx, v.x);
                        v.y = fmaf(K.hdt, fy, v.y);
                        v.z = fmaf(K.hdt, fz, v.z);
                    }
                    p.x = wrap_drift(fmaf(K.dt, v.x, p.x), g.L);
                    p.y = wrap_drift(fmaf(K.dt, v.y, p.y), g.L);
                    p.z = wrap_drift(fmaf(K.dt, v.z, p.z), g.L);
                    const int c = cell_id(cell_coord(p.x, g), cell_coord(p.y, g), cell_coord(p.z, g), g);
                    v.w = __int_as_float(atomicAdd(&cell_count[c], 1));   // rank inside the new cell
                    pos_out[myslot] = p;
                    vel[myslot] = v;
                }
            }
            if (ENERGY && myvalid) {
                // PE = 4 eps (A - B) - n ushift [+ f_rc sum(r - rc)],  W = 24 eps (2A - B) [- f_rc sum r]
                const double nin = (double)A.cnt.x + (double)A.cnt.y;
                const double sA = (double)A.sA.x + (double)A.sA.y, sB = (double)A.sB.x + (double)A.sB.y;
                pe_tot += dpe + P.eps4 * (sA - sB) - nin * P.ushift;
                w_tot += dw + P.eps24 * (2.0 * sA - sB);
                if (MODE2) {
                    pe_tot += P.f_rc * (double)A.sR;
                    w_tot -= P.f_rc * ((double)A.sR + nin * P.rc);
                }
            }
        }
    }
    if (ENERGY) {
        pe_tot = warp_sum(pe_tot);
        w_tot = warp_sum(w_tot);
        if (lane == 0) {
            const int u = (cx * n + cy) * n + cz;            // partials by linear cell number in either ordering
            part_pe[u] = 0.5 * pe_tot;                       // every pair is visited from both ends
            part_w[u] = 0.5 * w_tot;
        }
    }
}

// energy = false: forces only.  fused = true: the epilogue integrates (interior steps of md_step): reads and
// writes s->vel, writes the drifted positions to s->pos2 and the new cells' histogram to s->cell_count.
int ljmd_forces_cell3(md_sim *s, bool energy, bool fused)
{
    const Grid &g = s->grid;
    const dim3 grid = g.morton ? dim3((unsigned)g.nid, 1, 1) : dim3(g.n, g.n, g.n);
    if ((int64_t)g.ncells > s->part_cap) return MD_ENOMEM;
    double *ppe = s->part + (size_t)s->part_cap;
    double *pw = s->part + 2 * (size_t)s->part_cap;
    const PairParams &P = s->pp;
    F3Const K;
    memset(&K, 0, sizeof(K));
    const double rc2_lo = P.rc2 * (1.0 - 4e-6), rc2_hi = P.rc2 * (1.0 + 4e-6);
    const double p2 = fmin(P.precise_r2, rc2_lo);
    K.p2 = (float)p2;
    K.rc2_lo = (float)rc2_lo;
    K.mid = (float)(0.5 * (p2 + rc2_lo));
    K.hw = (float)(0.5 * (rc2_lo - p2));
    K.hw2 = (float)(rc2_hi - (double)K.mid);
    K.h = 0.5f * g.side;
    K.hd = (double)K.h;
    K.tile_exact = (1.5 * (double)g.last < 4.0 && (double)g.side >= 2.0) ? 1 : 0;
    // a candidate is kept when its distance to the home box is below rc (plus the FP32 rounding of the test)
    K.prune2 = (float)(rc2_hi + 1e-4);
    K.sig2 = P.sig2f;
    K.eps24 = P.eps24f;
    K.neps48 = -2.0f * P.eps24f;
    K.f_rcf = P.f_rcf;
    K.rcf = P.rcf;
    K.hdt = s->hdtf;
    K.dt = s->dtf;
    const int nmax = (int)s->N - 1;
#define F3_LAUNCH(M2, EN, FU) \
    k_fc3<M2, EN, FU><<<grid, 32, 0, s->stream>>>(s->pos, s->cell_start, g, P, K, s->frc, ppe, pw, nmax, s->vel, s->pos2, s->cell_count)
    if (P.mode == 2) {
        if (fused) { if (energy) F3_LAUNCH(true, true, true); else F3_LAUNCH(true, false, true); }
        else { if (energy) F3_LAUNCH(true, true, false); else F3_LAUNCH(true, false, false); }
    } else {
        if (fused) { if (energy) F3_LAUNCH(false, true, true); else F3_LAUNCH(false, false, true); }
        else { if (energy) F3_LAUNCH(false, true, false); else F3_LAUNCH(false, false, false); }
    }
#undef F3_LAUNCH
    CKL(s);
    ljmd_tick(s, TAG_FORCE);
    if (energy) s->n_pe = g.ncells;
    if (fused) s->fused_pending = true;
    return MD_OK;
}
