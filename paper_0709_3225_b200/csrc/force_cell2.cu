// Cell-list Lennard-Jones force, second generation (one block per
// cell, the atoms of its 27 neighbour cells staged through shared memory).  Same method as
// force_cell.cu (whose kernel stays as the neighbour-list builder and as a cross-check, option
// "cell_kernel" = 1): CSR cells, candidates staged in the frame of the warp's first cell (exact in
// FP32), FFMA2 ballot filter, per-lane walk over the hit bits, FP64 for the
// steep part of the potential.  What changed, each from an ncu finding on the first kernel
// (DESIGN.md section 7):
//   * the tile is SoA (x, y, z), |u|^2 is recomputed by the filter: 5.4 KB instead of 8.7 KB per warp,
//     24 instead of 16 resident warps;
//   * the filter takes row PAIRS (1..8), so a cell of 13 atoms filters 14 rows, not 16;
//   * the walk evaluates two hits per iteration with packed f32x2 arithmetic (FFMA2/FMUL2/FADD2),
//     takes its trip count from a popcount pre-pass (no vote per iteration), folds the validity of
//     a slot into the window predicate, and pushes FP64 candidates through a clamped pointer;
//   * staging looks its segment up from a byte label, one LDS per candidate;
//   * PE and the virial are only accumulated when the caller will read them (ENERGY).
#include <math.h>
#include "common.cuh"
#include "pair.cuh"

#ifndef F2_CAP
#define F2_CAP 416                    // staged candidates per pass (13 words; 27 cells of 13 atoms = 351)
#endif
#define F2_NW (F2_CAP / 32)
#define F2_QCAP 10                    // queued FP64 pairs per lane (row F2_QCAP is the overflow sentinel)
#ifndef F2_MINB
#define F2_MINB 20                    // resident one-warp blocks per SM
#endif
#define F2_FULL 0xffffffffu

template <int KK> struct F2Geom {
    static constexpr int NZ2 = KK + 2;                  // cells per staged z-run
    static constexpr int NSEG = 9 * NZ2;                // neighbour cells of the group
    static constexpr int NH = (NSEG + 31) / 32;         // segments per lane
    static constexpr int DSEG = NSEG;                   // dummy segment: far away, labels the padding
    static constexpr int NSEGP = (NSEG + 1 + 3) & ~3;
};

template <int KK> struct F2Smem {
    float t[3][32 + F2_CAP];          // candidate u = l + (origin offset) - centre; index 31 is readable (idle slots)
    unsigned msk[F2_NW][16];          // hit-mask words [32-candidate word][row]
    float4 seg[F2Geom<KK>::NSEGP];    // per segment: origin offset minus centre, (first slot - candidates before it)
    int seg_pref[F2Geom<KK>::NSEGP];  // candidates before segment k
    float rax[16], ray[16], raz[16], rT[16];   // filter rows: -2 u_i and threshold - |u_i|^2
    unsigned short q[F2_QCAP + 1][32];
    unsigned char lab[F2_CAP];        // segment of candidate c of the current pass
};

struct F2Const {
    float rc2_lo, rc2_thr, p2;        // FP32 window [p2, rc2_lo); filter threshold rc^2 (1 + 4e-6) + margin
    float sig2, eps24, neps48;
    float h;                          // half a cell side
    float f_rcf, rcf;                 // mode 2
    double hd;
    int nzu;
    int tile_exact;                   // the staged FP32 coordinates are exact for warps away from the box origin
    float hdt, dt;                    // fused integrator
};

__device__ __forceinline__ int f2_bfind(unsigned x)      // index of the highest set bit, -1 for 0
{
    int b;
    asm("bfind.u32 %0, %1;" : "=r"(b) : "r"(x));
    return b;
}

__device__ __forceinline__ unsigned f2_bit(int b)        // 1 << b, 0 for b = -1 (PTX shl clamps the amount)
{
    unsigned r;
    asm("shl.b32 %0, 1, %1;" : "=r"(r) : "r"(b));
    return r;
}

__device__ __forceinline__ float f2_rcp(float x)
{
    float y;
    asm("rcp.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x));
    return y;
}

// FP64 pair term without branches (two of them are interleaved per iteration of the FP64 queue): a pair
// with r^2 >= rc^2 (or an idle slot, which passes a far-away displacement) contributes exactly zero.
template <bool MODE2, bool ENERGY>
__device__ __forceinline__ void f2_pair64(const PairParams &P, double dx, double dy, double dz, double &fx,
                                          double &fy, double &fz, double &pe, double &w)
{
    const double r2 = fma(dx, dx, fma(dy, dy, dz * dz));
    const bool in = r2 < P.rc2;                          // strict
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

#define F2_TS ((32 + F2_CAP) * 4)     // byte stride between the x, y and z arrays of the tile

template <int OFF> __device__ __forceinline__ float f2_lds_f32(unsigned addr)
{
    float v;
    asm volatile("ld.shared.f32 %0, [%1+%2];" : "=f"(v) : "r"(addr), "n"(OFF));
    return v;
}

__device__ __forceinline__ unsigned f2_lds_u32(unsigned addr)
{
    unsigned v;
    asm volatile("ld.shared.u32 %0, [%1];" : "=r"(v) : "r"(addr));
    return v;
}

// Append the 16-bit tile offset `a` to the lane's FP64 queue when `push`; the write pointer stops at qend
// (the sentinel row), which marks an overflow.
__device__ __forceinline__ void f2_push(unsigned &qa, int a, bool push, unsigned qend)
{
    asm volatile("{ .reg .pred p;\n\t setp.ne.b32 p, %2, 0;\n\t @p st.shared.u16 [%0], %1;\n\t }"
                 :: "r"(qa), "h"((unsigned short)a), "r"((int)push) : "memory");
    qa = push ? min(qa + 64u, qend) : qa;
}

// Filter: lane = candidate, NP row pairs in registers (two rows per FFMA2); per (row, 32 candidates)
// 1.5 FFMA2 + compare + ballot.  r^2 - |u_i|^2 = |u_j|^2 - 2 u_i.u_j is compared with T_i.
template <int NP>
__device__ __forceinline__ void f2_filter(const float *__restrict__ tx, const float *__restrict__ ty,
                                          const float *__restrict__ tz, unsigned (*__restrict__ msk)[16],
                                          const float *__restrict__ rax, const float *__restrict__ ray,
                                          const float *__restrict__ raz, const float *__restrict__ rT,
                                          const int nsteps, const int lane)
{
    float2 ax[NP], ay[NP], az[NP], T[NP];
#pragma unroll
    for (int p = 0; p < NP; p++) {
        ax[p] = *reinterpret_cast<const float2 *>(&rax[2 * p]);
        ay[p] = *reinterpret_cast<const float2 *>(&ray[2 * p]);
        az[p] = *reinterpret_cast<const float2 *>(&raz[2 * p]);
        T[p] = *reinterpret_cast<const float2 *>(&rT[2 * p]);
    }
    for (int st = 0; st < nsteps; st++) {
        const int c = st * 32 + lane;
        const float x = tx[c], y = ty[c], z = tz[c];
        const float w = fmaf(x, x, fmaf(y, y, z * z));
        const float2 X = make_float2(x, x), Y = make_float2(y, y), Z = make_float2(z, z), W = make_float2(w, w);
        unsigned m[2 * NP];
#pragma unroll
        for (int p = 0; p < NP; p++) {
            const float2 v = __ffma2_rn(ax[p], X, __ffma2_rn(ay[p], Y, __ffma2_rn(az[p], Z, W)));
            m[2 * p] = __ballot_sync(F2_FULL, v.x < T[p].x);
            m[2 * p + 1] = __ballot_sync(F2_FULL, v.y < T[p].y);
        }
        // one lane stores (a 16-byte store of the same value by all lanes costs four wavefronts, not one)
        if (lane == 0) {
#pragma unroll
            for (int q = 0; q < NP / 2; q++)
                *reinterpret_cast<uint4 *>(&msk[st][4 * q]) = make_uint4(m[4 * q], m[4 * q + 1], m[4 * q + 2], m[4 * q + 3]);
            if (NP & 1) *reinterpret_cast<uint2 *>(&msk[st][2 * (NP - 1)]) = make_uint2(m[2 * (NP - 1)], m[2 * NP - 1]);
        }
    }
}

// FUSED: the lane that owns F_i also applies the closing half-kick of this step and the opening half-kick,
// drift, wrap and cell histogram of the next one (the arithmetic of k_kick_drift_bin3<2>, cells.cu, on the
// float force), writing the drifted positions to pos_out and the kicked velocities (rank in .w) in place:
// an interior step of md_step is then force kernel + scan + scatter, and the forces never reach HBM.
template <int KK, bool MODE2, bool ENERGY, bool FUSED>
__global__ void __launch_bounds__(32, F2_MINB)
k_fc2(const float4 *__restrict__ lpos, const int *__restrict__ cell_start, const Grid g, const PairParams P,
      const F2Const K, float4 *__restrict__ frc, double *__restrict__ part_pe, double *__restrict__ part_w,
      const int nmax, const float4 *__restrict__ pos, float4 *__restrict__ vel, float4 *__restrict__ pos_out,
      int *__restrict__ cell_count)
{
    typedef F2Geom<KK> G;
    __shared__ __align__(16) F2Smem<KK> S;
    const int lane = threadIdx.x;
    const int n = g.n;
    const int zu = blockIdx.x, cy = blockIdx.y, cx = blockIdx.z;
    const int z0 = zu * KK;
    const int kk = min(KK, n - z0);
    const int cfirst = (cx * n + cy) * n + z0;
    double pe_tot = 0.0, w_tot = 0.0;
    {
        // ---- the 9 x (KK + 2) neighbour cells ("segments"): first slot, count, exact origin offset.
        // Their cell_start loads do not wait for the group's own (issued below, tested after).
        const float hz = 0.5f * (float)kk * g.side;              // centre of the group in the frame of its first cell
        // no staged cell has index 0 in any dimension: every global coordinate is >= side >= 2
        const bool exact = K.tile_exact && cx >= 2 && cx <= n - 2 && cy >= 2 && cy <= n - 2 && z0 >= 2 && z0 + kk <= n - 1;
        int cnt[G::NH], start[G::NH], incl[G::NH];
        float ox[G::NH], oy[G::NH], oz[G::NH];
#pragma unroll
        for (int h = 0; h < G::NH; h++) {
            const int sgi = lane + 32 * h;                        // segment = (column, dz)
            cnt[h] = 0; start[h] = 0; ox[h] = oy[h] = oz[h] = 0.f;
            const int col = sgi / G::NZ2, dz = sgi - col * G::NZ2 - 1;     // dz = -1 .. KK
            if (sgi < G::NSEG && dz <= kk) {
                const int ax = col / 3 - 1, ay = col - (col / 3) * 3 - 1;
                int nx = cx + ax, ny = cy + ay, nz = z0 + dz;
                nx += (nx < 0) ? n : 0; nx -= (nx >= n) ? n : 0;
                ny += (ny < 0) ? n : 0; ny -= (ny >= n) ? n : 0;
                nz += (nz < 0) ? n : 0; nz -= (nz >= n) ? n : 0;
                // distance between the cell origins: exact
                ox[h] = (ax == 0) ? 0.f : (ax > 0 ? ((cx == n - 1) ? g.last : g.side) : -((nx == n - 1) ? g.last : g.side));
                oy[h] = (ay == 0) ? 0.f : (ay > 0 ? ((cy == n - 1) ? g.last : g.side) : -((ny == n - 1) ? g.last : g.side));
                if (dz < 0) oz[h] = -((nz == n - 1) ? g.last : g.side);
                else oz[h] = (float)dz * g.side + ((dz > 0 && z0 + dz - 1 == n - 1) ? (g.last - g.side) : 0.f);
                const int nb = (nx * n + ny) * n + nz;
                start[h] = cell_start[nb];
                cnt[h] = cell_start[nb + 1] - start[h];
            }
        }
        const int ibeg = cell_start[cfirst], ni = cell_start[cfirst + kk] - ibeg;
        if (ni > 0) {
        int carry = 0;
#pragma unroll
        for (int h = 0; h < G::NH; h++) {
            int v = cnt[h];
#pragma unroll
            for (int o = 1; o < 32; o <<= 1) {
                const int y = __shfl_up_sync(F2_FULL, v, o);
                if (lane >= o) v += y;
            }
            incl[h] = v + carry;
            carry += __shfl_sync(F2_FULL, v, 31);
        }
        const int total = carry;
#pragma unroll
        for (int h = 0; h < G::NH; h++) {
            const int sgi = lane + 32 * h;
            if (sgi < G::NSEG) {
                const int pref = incl[h] - cnt[h];
                S.seg_pref[sgi] = pref;
                S.seg[sgi] = make_float4(ox[h] - K.h, oy[h] - K.h, oz[h] - hz, __int_as_float(start[h] - pref));
            }
        }
        if (lane == 0) {
            S.seg[G::DSEG] = make_float4(1.0e4f, 1.0e4f, 1.0e4f, __int_as_float(0));
            S.t[0][31] = S.t[1][31] = S.t[2][31] = 1.0e4f;
        }
        __syncwarp();
        const int cself0 = S.seg_pref[4 * G::NZ2 + 1];           // candidate index of the group's own atom 0
        const float *tx = &S.t[0][32], *ty = &S.t[1][32], *tz = &S.t[2][32];
        int staged_t0 = -1;

        for (int i0 = 0; i0 < ni; i0 += 16) {
            // ---- lanes of this pass: nrow atoms, SL slices of the mask words per atom
            const int nrow = min(16, ni - i0);
            const float invrow = __frcp_rn((float)nrow);
            const int SL = (int)(32.25f * invrow);
            const int sl = (int)(((float)lane + 0.5f) * invrow), li_ = lane - sl * nrow;
            const bool myvalid = sl < SL;
            const int myslot = ibeg + i0 + li_;
            const float4 lme = lpos[myslot];
            float4 pme4, vme4;
            if (FUSED) { pme4 = pos[myslot]; vme4 = vel[myslot]; }   // early: the latency hides behind the pass
            float zoff_me = 0.f;
#pragma unroll
            for (int k = 1; k < KK; k++) zoff_me += (k < kk && myslot >= cell_start[cfirst + k]) ? g.side : 0.f;
            const float ux = lme.x - K.h, uy = lme.y - K.h, uz = (lme.z + zoff_me) - hz;
            // rows of the filter (lanes of slice 0 are the rows; the rest up to 16 never hit)
            __syncwarp();
            if (lane < 16) {
                const bool real = lane < nrow;
                S.rax[lane] = real ? -2.f * ux : 0.f;
                S.ray[lane] = real ? -2.f * uy : 0.f;
                S.raz[lane] = real ? -2.f * uz : 0.f;
                S.rT[lane] = real ? K.rc2_thr - fmaf(ux, ux, fmaf(uy, uy, uz * uz)) : -INFINITY;
            }
            for (int t0 = 0; t0 < total; t0 += F2_CAP) {
                const int cnt_p = min(F2_CAP, total - t0);
                const int nsteps = (cnt_p + 31) >> 5;
                if (t0 != staged_t0) {
                    // ---- stage candidates t0 .. t0 + cnt_p of the concatenated neighbour cells
                    staged_t0 = t0;
                    __syncwarp();
#pragma unroll
                    for (int h = 0; h < G::NH; h++) {             // every lane labels the candidates of its segments
                        const int pref = incl[h] - cnt[h];
                        const int lo = max(pref, t0) - t0, hi = min(pref + cnt[h], t0 + cnt_p) - t0;
                        for (int c = lo; c < hi; c++) S.lab[c] = (unsigned char)(lane + 32 * h);
                    }
                    if (cnt_p + lane < nsteps * 32) S.lab[cnt_p + lane] = (unsigned char)G::DSEG;
                    __syncwarp();
                    for (int c0 = lane; c0 < nsteps * 32; c0 += 128) {
                        float4 l[4], sg[4];
#pragma unroll
                        for (int u = 0; u < 4; u++) {
                            const int c = c0 + 32 * u;
                            sg[u] = S.seg[(c < nsteps * 32) ? S.lab[c] : G::DSEG];
                        }
#pragma unroll
                        for (int u = 0; u < 4; u++) {
                            const int c = c0 + 32 * u;
                            l[u] = lpos[min(__float_as_int(sg[u].w) + t0 + c, nmax)];
                        }
#pragma unroll
                        for (int u = 0; u < 4; u++) {
                            const int c = c0 + 32 * u;
                            if (c < nsteps * 32) {
                                S.t[0][32 + c] = l[u].x + sg[u].x;
                                S.t[1][32 + c] = l[u].y + sg[u].y;
                                S.t[2][32 + c] = l[u].z + sg[u].z;
                            }
                        }
                    }
                }
                __syncwarp();
#ifndef F2_SKIP_FILTER
                switch ((nrow + 1) >> 1) {
                case 1: f2_filter<1>(tx, ty, tz, S.msk, S.rax, S.ray, S.raz, S.rT, nsteps, lane); break;
                case 2: f2_filter<2>(tx, ty, tz, S.msk, S.rax, S.ray, S.raz, S.rT, nsteps, lane); break;
                case 3: f2_filter<3>(tx, ty, tz, S.msk, S.rax, S.ray, S.raz, S.rT, nsteps, lane); break;
                case 4: f2_filter<4>(tx, ty, tz, S.msk, S.rax, S.ray, S.raz, S.rT, nsteps, lane); break;
                case 5: f2_filter<5>(tx, ty, tz, S.msk, S.rax, S.ray, S.raz, S.rT, nsteps, lane); break;
                case 6: f2_filter<6>(tx, ty, tz, S.msk, S.rax, S.ray, S.raz, S.rT, nsteps, lane); break;
                case 7: f2_filter<7>(tx, ty, tz, S.msk, S.rax, S.ray, S.raz, S.rT, nsteps, lane); break;
                default: f2_filter<8>(tx, ty, tz, S.msk, S.rax, S.ray, S.raz, S.rT, nsteps, lane); break;
                }
#endif
                __syncwarp();
                // the pair (i, i) is not a pair
                if (lane < nrow) {
                    const int cs = cself0 + i0 + lane - t0;
                    if (cs >= 0 && cs < cnt_p) S.msk[cs >> 5][lane] &= ~(1u << (cs & 31));
                }
                __syncwarp();
                // ---- pre-pass: hits and iterations of my words st = sl, sl + SL, ...
                int nhit = 0, iters = 0;
                if (myvalid)
                    for (int st = sl; st < nsteps; st += SL) {
                        const int p = __popc(S.msk[st][li_]);
                        nhit += p;
                        iters += max(1, (p + 1) >> 1);
                    }
#ifdef F2_SKIP_WALK
                const int niter = 0;
#else
                const int niter = __reduce_max_sync(F2_FULL, iters);
#endif
                // ---- walk: two hits per iteration; an exhausted slot reads the entry before its word
                // (any valid entry) and is masked through the window predicate.  ca = byte offset of
                // candidate (word, bit 0) in the tile arrays; a queued pair is remembered by that offset.
                const unsigned mbase = (unsigned)__cvta_generic_to_shared(&S.msk[0][0]);
                const unsigned mend = mbase + (unsigned)nsteps * 64u;
                unsigned ma = (myvalid && sl < nsteps) ? mbase + (unsigned)(sl * 16 + li_) * 4u : mend;
                const unsigned mstride = (unsigned)SL * 64u;
                const int cstride = SL * 128;
                unsigned cur = 0u;
                int ca = sl * 128;
                if (ma < mend) { cur = f2_lds_u32(ma); ma += mstride; } else ca = 0;
                const unsigned tb = (unsigned)__cvta_generic_to_shared(tx);
                const unsigned q0 = (unsigned)__cvta_generic_to_shared(&S.q[0][lane]);
                unsigned qa = q0;
                const unsigned qend = q0 + F2_QCAP * 64u;
                float2 fx2 = make_float2(0.f, 0.f), fy2 = fx2, fz2 = fx2, sA2 = fx2, sB2 = fx2;
                float sR = 0.f;
                const float2 one2 = make_float2(1.f, 1.f), sig22 = make_float2(K.sig2, K.sig2);
                const float2 e24 = make_float2(K.eps24, K.eps24), ne48 = make_float2(K.neps48, K.neps48);
                const float2 nUX = make_float2(-ux, -ux), nUY = make_float2(-uy, -uy), nUZ = make_float2(-uz, -uz);
                for (int it = 0; it < niter; it++) {
                    const int b0 = f2_bfind(cur);
                    cur &= ~f2_bit(b0);
                    const int b1 = f2_bfind(cur);
                    cur &= ~f2_bit(b1);
                    const int a0 = ca + 4 * b0, a1 = ca + 4 * b1;
                    const float2 X = make_float2(f2_lds_f32<0>(tb + a0), f2_lds_f32<0>(tb + a1));
                    const float2 Y = make_float2(f2_lds_f32<F2_TS>(tb + a0), f2_lds_f32<F2_TS>(tb + a1));
                    const float2 Z = make_float2(f2_lds_f32<2 * F2_TS>(tb + a0), f2_lds_f32<2 * F2_TS>(tb + a1));
                    if (cur == 0u && ma < mend) {
                        cur = f2_lds_u32(ma);
                        ma += mstride;
                        ca += cstride;
                    }
                    const float2 dx = __fadd2_rn(X, nUX), dy = __fadd2_rn(Y, nUY), dz = __fadd2_rn(Z, nUZ);
                    const float2 r2 = __ffma2_rn(dx, dx, __ffma2_rn(dy, dy, __fmul2_rn(dz, dz)));
                    // p2 <= r2 < rc2_lo: FP32 term.  Everything else the filter let through (the steep
                    // part, the sliver around rc^2, false positives beyond it) goes to the FP64 queue.
                    const bool v0 = b0 >= 0, v1 = b1 >= 0;
                    const bool in0 = v0 && r2.x >= K.p2 && r2.x < K.rc2_lo;
                    const bool in1 = v1 && r2.y >= K.p2 && r2.y < K.rc2_lo;
                    f2_push(qa, a0, v0 && !in0, qend);
                    f2_push(qa, a1, v1 && !in1, qend);
                    float2 inv = make_float2(f2_rcp(r2.x), f2_rcp(r2.y));
                    inv = __ffma2_rn(inv, __ffma2_rn(make_float2(-r2.x, -r2.y), inv, one2), inv);   // one Newton step
                    // a slot outside the FP32 window contributes nothing: 1/r^2 := 0 (also swallows the inf/NaN
                    // of an exhausted slot that happened to read the atom itself)
                    inv.x = in0 ? inv.x : 0.f;
                    inv.y = in1 ? inv.y : 0.f;
                    const float2 s2 = __fmul2_rn(sig22, inv);
                    const float2 s6 = __fmul2_rn(__fmul2_rn(s2, s2), s2);
                    // -f/r = inv s6 (24 eps - 48 eps s6)
                    float2 nfr = __fmul2_rn(__fmul2_rn(inv, s6), __ffma2_rn(ne48, s6, e24));
                    if (MODE2) {
                        const float r0 = sqrtf(r2.x), r1 = sqrtf(r2.y);
                        nfr.x += in0 ? K.f_rcf * inv.x * r0 : 0.f;
                        nfr.y += in1 ? K.f_rcf * inv.y * r1 : 0.f;
                        if (ENERGY) {
                            sR += in0 ? (r0 - K.rcf) : 0.f;
                            sR += in1 ? (r1 - K.rcf) : 0.f;
                        }
                    }
                    fx2 = __ffma2_rn(nfr, dx, fx2);
                    fy2 = __ffma2_rn(nfr, dy, fy2);
                    fz2 = __ffma2_rn(nfr, dz, fz2);
                    if (ENERGY) {
                        sA2 = __ffma2_rn(s6, s6, sA2);
                        sB2 = __fadd2_rn(sB2, s6);
                    }
                }
                // ---- FP64 part of this pass: queued pairs from the exact local coordinates; a lane whose
                // queue overflowed rescans its words and takes every pair outside the FP32 window
                double dfx = 0.0, dfy = 0.0, dfz = 0.0, dpe = 0.0, dw = 0.0;
                int ncl;
                {
                    const bool ovf = qa == qend;
                    const int nq = ovf ? 0 : (int)(qa - q0) >> 6;
                    ncl = nq;
                    const double zme = (double)hz - (double)zoff_me;
                    // exact displacement of staged candidate c from my atom.  Away from the box origin the
                    // staged FP32 coordinates are exact (multiples of 2^-22 below 4: DESIGN.md section 5) and
                    // their difference is the displacement; otherwise it is rebuilt from the cell-local
                    // coordinates and the exact origin offset of the candidate's cell.
                    auto disp = [&](const int c, double &ex, double &ey, double &ez) {
                        if (exact) {
                            ex = (double)tx[c] - (double)ux;
                            ey = (double)ty[c] - (double)uy;
                            ez = (double)tz[c] - (double)uz;
                        } else {
                            const float4 lme = lpos[myslot];
                            const float4 sg = S.seg[S.lab[c]];
                            const float4 lj = lpos[min(__float_as_int(sg.w) + t0 + c, nmax)];
                            ex = ((double)lj.x - (double)lme.x) + ((double)sg.x + K.hd);
                            ey = ((double)lj.y - (double)lme.y) + ((double)sg.y + K.hd);
                            ez = ((double)lj.z - (double)lme.z) + ((double)sg.z + zme);
                        }
                    };
#ifdef F2_SKIP_FP64
                    const int maxq = 0;
#else
                    const int maxq = __reduce_max_sync(F2_FULL, nq);
#endif
                    for (int k = 0; k < maxq; k += 2) {          // two independent chains per iteration
                        // an idle slot takes candidate -1: the far-away entry in front of the tile
                        const int ca_ = (k < nq) ? (int)S.q[k][lane] >> 2 : -1;
                        const int cb_ = (k + 1 < nq) ? (int)S.q[k + 1][lane] >> 2 : -1;
                        double ax_, ay_, az_, bx_, by_, bz_;
                        if (exact) {
                            disp(ca_, ax_, ay_, az_);
                            disp(cb_, bx_, by_, bz_);
                        } else {
                            ax_ = ay_ = az_ = bx_ = by_ = bz_ = 1.0e4;
                            if (ca_ >= 0) disp(ca_, ax_, ay_, az_);
                            if (cb_ >= 0) disp(cb_, bx_, by_, bz_);
                        }
                        f2_pair64<MODE2, ENERGY>(P, ax_, ay_, az_, dfx, dfy, dfz, dpe, dw);
                        f2_pair64<MODE2, ENERGY>(P, bx_, by_, bz_, dfx, dfy, dfz, dpe, dw);
                    }
                    if (__any_sync(F2_FULL, ovf)) {
                        if (ovf) {
                            ncl = 0;
                            for (int st = sl; st < nsteps; st += SL) {
                                unsigned m = S.msk[st][li_];
                                while (m) {
                                    const int b = __ffs(m) - 1;
                                    m &= m - 1u;
                                    const int c = st * 32 + b;
                                    const float ddx = tx[c] - ux, ddy = ty[c] - uy, ddz = tz[c] - uz;
                                    const float rr = fmaf(ddx, ddx, fmaf(ddy, ddy, ddz * ddz));
                                    if (!(rr >= K.p2 && rr < K.rc2_lo)) {
                                        ncl++;
                                        double ex, ey, ez;
                                        disp(c, ex, ey, ez);
                                        f2_pair64<MODE2, ENERGY>(P, ex, ey, ez, dfx, dfy, dfz, dpe, dw);
                                    }
                                }
                            }
                        }
                    }
                }
                // ---- totals of this lane, reduction over the slices of an atom, store (a later candidate
                // pass adds to what the earlier ones stored)
                double tx_ = dfx + (double)fx2.x + (double)fx2.y;
                double ty_ = dfy + (double)fy2.x + (double)fy2.y;
                double tz_ = dfz + (double)fz2.x + (double)fz2.y;
                double ox_ = 0.0, oy_ = 0.0, oz_ = 0.0;
                for (int k = 1; k < SL; k++) {
                    const int src = lane + k * nrow;               // < 32 for the lanes of slice 0
                    ox_ += __shfl_sync(F2_FULL, tx_, src);
                    oy_ += __shfl_sync(F2_FULL, ty_, src);
                    oz_ += __shfl_sync(F2_FULL, tz_, src);
                }
                if (sl == 0) {
                    if (t0 > 0) {
                        const float4 f0 = frc[myslot];
                        tx_ += (double)f0.x; ty_ += (double)f0.y; tz_ += (double)f0.z;
                    }
                    const float fx = (float)(tx_ + ox_), fy = (float)(ty_ + oy_), fz = (float)(tz_ + oz_);
                    if (!FUSED || t0 + F2_CAP < total) {
                        frc[myslot] = make_float4(fx, fy, fz, 0.f);
                    } else {
                        float4 p = pme4, v = vme4;
#pragma unroll
                        for (int k = 0; k < 2; k++) {
                            v.x = fmaf(K.hdt, fx, v.x);
                            v.y = fmaf(K.hdt, fy, v.y);
                            v.z = fmaf(K.hdt, fz, v.z);
                        }
                        p.x = wrap_drift(fmaf(K.dt, v.x, p.x), g.L);
                        p.y = wrap_drift(fmaf(K.dt, v.y, p.y), g.L);
                        p.z = wrap_drift(fmaf(K.dt, v.z, p.z), g.L);
                        const int c = (cell_coord(p.x, g) * n + cell_coord(p.y, g)) * n + cell_coord(p.z, g);
                        v.w = __int_as_float(atomicAdd(&cell_count[c], 1));   // rank inside the new cell
                        pos_out[myslot] = p;
                        vel[myslot] = v;
                    }
                }
                if (ENERGY) {
                    // PE = 4 eps (A - B) - n ushift [+ f_rc sum(r - rc)],  W = 24 eps (2A - B) [- f_rc sum r]
                    const int nin = nhit - ncl;
                    const double sA = (double)sA2.x + (double)sA2.y, sB = (double)sB2.x + (double)sB2.y;
                    pe_tot += dpe + P.eps4 * (sA - sB) - (double)nin * P.ushift;
                    w_tot += dw + P.eps24 * (2.0 * sA - sB);
                    if (MODE2) {
                        pe_tot += P.f_rc * (double)sR;
                        w_tot -= P.f_rc * ((double)sR + (double)nin * P.rc);
                    }
                }
            }
        }
    }
    }
    if (ENERGY) {
        pe_tot = warp_sum(pe_tot);
        w_tot = warp_sum(w_tot);
        if (lane == 0) {
            const int u = (cx * n + cy) * K.nzu + zu;
            part_pe[u] = 0.5 * pe_tot;                       // every pair is visited from both ends
            part_w[u] = 0.5 * w_tot;
        }
    }
}

// Cells per row group (warp): option "cell_group", else from the mean occupancy.
int ljmd_fc2_group_cells(const md_sim *s, const Grid &g)
{
    int kz = s->cell_group;
    if (kz <= 0) {
        const double occ = (double)s->N / (double)g.ncells;
        kz = (occ >= 9.0) ? 1 : (occ >= 5.5 ? 2 : 3);
    }
    if (kz == 4) kz = 3;
    if (kz > 5) kz = 5;
    if (kz < 1 || g.n < 8) kz = 1;                  // dz * side must stay exact in FP32 (L >= 16)
    return kz;
}

template <int KK>
static void fc2_launch(md_sim *s, const Grid &g, const dim3 grid, const F2Const &K, double *ppe, double *pw, bool energy, bool fused)
{
    const PairParams &P = s->pp;
    const int nmax = (int)s->N - 1;
#define F2_LAUNCH(M2, EN, FU) \
    k_fc2<KK, M2, EN, FU><<<grid, 32, 0, s->stream>>>(s->lpos, s->cell_start, g, P, K, s->frc, ppe, pw, nmax, s->pos, s->vel, s->pos2, s->cell_count)
    if (fused) {                                    // interior steps: forces only
        if (P.mode == 2) F2_LAUNCH(true, false, true); else F2_LAUNCH(false, false, true);
    } else if (P.mode == 2) {
        if (energy) F2_LAUNCH(true, true, false); else F2_LAUNCH(true, false, false);
    } else {
        if (energy) F2_LAUNCH(false, true, false); else F2_LAUNCH(false, false, false);
    }
#undef F2_LAUNCH
}

// energy = false: forces only (interior steps of md_step, whose PE and virial nobody can read)
int ljmd_forces_cell2(md_sim *s, bool energy, bool fused)
{
    return ljmd_forces_cell2_on(s, s->grid, 0.0, energy, fused);
}

// The same kernel on any cell grid whose lpos/cell_start are current.  `stray`: how far an atom may sit outside
// its cell (skin cells between rebuilds, verlet.cu: half the skin); it widens the filter's rounding margin.
int ljmd_forces_cell2_on(md_sim *s, const Grid &g, double stray, bool energy, bool fused)
{
    if (fused) energy = false;
    const int kz = ljmd_fc2_group_cells(s, g);
    const int nzu = (g.n + kz - 1) / kz;
    const dim3 grid(nzu, g.n, g.n);
    const int64_t nunits = (int64_t)nzu * g.n * g.n;
    if (nunits > s->part_cap) return MD_ENOMEM;
    double *ppe = s->part + (size_t)s->part_cap;
    double *pw = s->part + 2 * (size_t)s->part_cap;
    const PairParams &P = s->pp;
    F2Const K;
    memset(&K, 0, sizeof(K));
    K.rc2_lo = (float)(P.rc2 * (1.0 - 4e-6));
    // Row groups of several cells stage candidates up to 3.5 cell sides from the frame centre, where
    // atoms whose global coordinate is below 4 (8 for kz = 5) lose up to 2.4e-7 (4.8e-7) of their
    // offset to FP32 rounding; the FP64 window is widened to r^2 < 1.5 sigma^2 so that every pair
    // with |df/dr| > 5 is still evaluated from the exact coordinates.
    double p2 = P.precise_r2;
    if ((kz > 1 || stray > 0.0) && !s->precise_r2_user) p2 = fmax(p2, 1.5 * P.sig2);
    K.p2 = (float)fmin(p2, 3.0e38);
    K.h = 0.5f * g.side;
    K.hd = (double)K.h;
    K.nzu = nzu;
    K.tile_exact = (kz == 1 && stray == 0.0 && 1.5 * (double)g.last < 4.0 && (double)g.side >= 2.0) ? 1 : 0;
    // farthest staged candidate from the frame centre, per dimension; FP32 rounding of the expanded form
    const double reach_xy = 1.5 * (double)g.last + stray, reach_z = (0.5 * kz + 1.0) * (double)g.last + stray;
    K.rc2_thr = (float)(P.rc2 * (1.0 + 4e-6) + 4.0e-6 * (2.0 * reach_xy * reach_xy + reach_z * reach_z) + 1e-6 * P.rc2);
    K.sig2 = P.sig2f;
    K.eps24 = P.eps24f;
    K.neps48 = -2.0f * P.eps24f;
    K.f_rcf = P.f_rcf;
    K.rcf = P.rcf;
    K.hdt = s->hdtf;
    K.dt = s->dtf;
    switch (kz) {
    case 1: fc2_launch<1>(s, g, grid, K, ppe, pw, energy, fused); break;
    case 2: fc2_launch<2>(s, g, grid, K, ppe, pw, energy, fused); break;
    case 3: fc2_launch<3>(s, g, grid, K, ppe, pw, energy, fused); break;
    default: fc2_launch<5>(s, g, grid, K, ppe, pw, energy, fused); break;
    }
    CKL(s);
    ljmd_tick(s, TAG_FORCE);
    if (energy) s->n_pe = (int)nunits;
    if (fused) s->fused_pending = true;
    return MD_OK;
}
