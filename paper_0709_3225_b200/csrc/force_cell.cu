// Cell-list Lennard-Jones force.  PAPER.md:112: one block (here: one
// warp) per cell, the atoms of its 27 neighbour cells staged through shared memory.
// What differs from the paper's G80 kernel (DESIGN.md sections 6, 7, 10):
//   * CSR cells from the counting sort instead of 32 placeholders with virtual particles;
//   * a warp owns a "row group" of 1..4 consecutive cells of one z-column (1 when cells hold about
//     13 atoms, more when they are sparsely filled); its candidates, the 9 x (cells + 2) cells
//     around it, are staged once in the frame of the group's first cell, u = l + (offset between
//     the cell origins) - centre, exact in FP32 on the power-of-two aligned grid;
//   * the distance test is a FILTER, 3 FFMA + compare + ballot per (atom i, 32 candidates):
//     lane = candidate (registers), the group's atoms two per FFMA2 in registers,
//     r^2 - |u_i|^2 = |u_j|^2 - 2 u_i.u_j against rc^2 + margin - |u_i|^2.  The ballot is the
//     i-major hit-mask word, stored to shared memory four rows per 16-byte store;
//   * evaluation: lane = (atom i, slice of its mask words); every lane walks its own hit bits,
//     two per iteration, so only the 15 % of candidates inside rc reach the pair term;
//   * mixed precision: pairs with r^2 < precise_r2 (default 1.3 sigma^2, the steep part of the
//     potential) or within 4e-6 of rc^2 are queued and evaluated in FP64 from the exact local
//     coordinates, the rest in FP32 with a Newton-corrected reciprocal; sums of s^6 and s^12
//     give PE and the virial.
// Tiles over candidates (FC_CAP per pass) and over atoms (16 per pass): any occupancy works.
#include <math.h>
#include "common.cuh"
#include "pair.cuh"

#ifndef FC_WARPS
#define FC_WARPS 1                    // warps (row groups) per block: a block retires with its warp, no idle slots (7 % faster than 2 or 4)
#endif
#define FC_T (FC_WARPS * 32)
#ifndef FC_CAP
#define FC_CAP 544                    // staged candidates per pass (27 list cells of 18.5 atoms fit)
#endif
#define FC_STEPS (FC_CAP / 32)
#define FC_CLOSE 8                    // queued FP64 pairs per lane
#ifndef FC_KZ_MAX
#define FC_KZ_MAX 5                   // cells per row group
#endif
#define FC_NSEG ((9 * (FC_KZ_MAX + 2) + 2 + 3) & ~3)   // multiple of 4: keeps the arrays behind it 16-byte aligned
#ifndef FC_MINB
#define FC_MINB 16                    // blocks per SM: 16 resident warps of 128 registers
#endif
#define FULLMASK 0xffffffffu

struct FcWarp {
    float4 tile[FC_CAP + 1];          // [FC_CAP] = dummy far-away entry for idle slots; candidate in the centre cell's frame; w = |u|^2 with the neighbour
                                      // segment number (0..53) in its 6 low mantissa bits
    unsigned msk[FC_STEPS][16];       // hit-mask words [32-candidate step][atom i of the pass]
    unsigned short close[FC_CLOSE][32];
    float4 seg[FC_NSEG];              // per segment (neighbour cell): origin offset minus h (x, y, z) and, as int
                                      // bits, (first slot - candidates before the cell)
    int seg_pref[FC_NSEG];            // candidates before segment k; [nseg ..] = total
    int seg_code[FC_NSEG];            // list mode: x/y offset code (kx + 5 ky) | (dz + 1) << 8 of segment k
    float rax[16], ray[16], raz[16], rT[16];   // filter rows: -2 u_i and threshold - |u_i|^2
};

struct FcConst {
    float rc2_lo, rc2_hi, p2, thr_margin, sig2, eps24, eps48, h;   // [rc2_lo, rc2_hi): decided in FP64
    double hd;
    int kz, nzu;                      // cells per row group, row groups per z-column
};

struct FcList {                       // neighbour-list output of the list mode (verlet.cu)
    unsigned *list;                   // [cap][npad]: slot of j | offset-table index << 23
    int *count;                       // [N]
    int *overflow;                    // set when a list is longer than cap
    int npad, cap;
};

struct FcGroup {                      // one warp's row group
    int ibeg, ni, total, kk, cfirst;  // first slot, atoms, candidates, cells, first cell
    float hz, side;                   // z centre of the group in the frame of its first cell
    double hzd;
    int pref0, cnt0, pref1, cnt1;     // this lane's two segments (lane, lane + 32)
    int z0, n;                        // first cell's z index, cells per dimension (list mode)
};

// z offset of row atom `slot` inside the group: (its cell - first cell) * side, exact
__device__ __forceinline__ float fc_row_zoff(const int *__restrict__ cell_start, const FcGroup &G, int slot)
{
    int q = 0;
    for (int k = 1; k < G.kk; k++) q += (slot >= cell_start[G.cfirst + k]) ? 1 : 0;
    return (float)q * G.side;
}

__device__ __forceinline__ float fc_rcp(float x)      // 1/x, x normal and positive: MUFU + one Newton step
{
    float y;
    asm("rcp.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x));
    const float e = fmaf(-x, y, 1.f);
    return fmaf(y, e, y);
}

__device__ __forceinline__ int fc_top_bit(unsigned x)      // index of the highest set bit (x != 0): one FLO
{
    int b;
    asm("bfind.u32 %0, %1;" : "=r"(b) : "r"(x));
    return b;
}

// FP64 pair term of my atom (exact local coordinates lme) with staged candidate c of pass t0
__device__ __forceinline__ void fc_precise(const FcWarp &S, const float4 *__restrict__ lpos, const PairParams &P,
                                           const FcConst &K, const float4 &lme, const double zme, int t0, int c,
                                           double &fx, double &fy, double &fz, double &pe, double &w)
{
    const float4 sg = S.seg[__float_as_int(S.tile[c].w) & 63];
    const float4 lj = lpos[__float_as_int(sg.w) + t0 + c];
    const double ex = ((double)lj.x - (double)lme.x) + ((double)sg.x + K.hd);
    const double ey = ((double)lj.y - (double)lme.y) + ((double)sg.y + K.hd);
    const double ez = ((double)lj.z - (double)lme.z) + ((double)sg.z + zme);     // zme = hz - my z offset
    pair_f64(P, ex, ey, ez, fx, fy, fz, pe, w);
}

// Filter: lane = candidate, rows = 4 NQ atoms (two per FFMA2), 3 FFMA + compare + ballot per
// (atom, 32 candidates); the ballots of four rows go to shared memory as one 16-byte store
// (every lane writes the same value).
template <int NQ>
__device__ __forceinline__ void fc_filter(FcWarp &S, const int nsteps, const int lane)
{
    float2 ax[2 * NQ], ay[2 * NQ], az[2 * NQ];
    float4 T[NQ];
#pragma unroll
    for (int q = 0; q < NQ; q++) {
        const float4 a = *reinterpret_cast<const float4 *>(&S.rax[4 * q]);
        const float4 b = *reinterpret_cast<const float4 *>(&S.ray[4 * q]);
        const float4 c = *reinterpret_cast<const float4 *>(&S.raz[4 * q]);
        ax[2 * q] = make_float2(a.x, a.y); ax[2 * q + 1] = make_float2(a.z, a.w);
        ay[2 * q] = make_float2(b.x, b.y); ay[2 * q + 1] = make_float2(b.z, b.w);
        az[2 * q] = make_float2(c.x, c.y); az[2 * q + 1] = make_float2(c.z, c.w);
        T[q] = *reinterpret_cast<const float4 *>(&S.rT[4 * q]);
    }
    for (int st = 0; st < nsteps; st++) {
        const float4 uj = S.tile[st * 32 + lane];
        const float2 X = make_float2(uj.x, uj.x), Y = make_float2(uj.y, uj.y), Z = make_float2(uj.z, uj.z),
                     W = make_float2(uj.w, uj.w);
#pragma unroll
        for (int q = 0; q < NQ; q++) {
            const float2 v0 = __ffma2_rn(ax[2 * q], X, __ffma2_rn(ay[2 * q], Y, __ffma2_rn(az[2 * q], Z, W)));
            const float2 v1 = __ffma2_rn(ax[2 * q + 1], X, __ffma2_rn(ay[2 * q + 1], Y, __ffma2_rn(az[2 * q + 1], Z, W)));
            uint4 m;
            m.x = __ballot_sync(FULLMASK, v0.x < T[q].x);
            m.y = __ballot_sync(FULLMASK, v0.y < T[q].y);
            m.z = __ballot_sync(FULLMASK, v1.x < T[q].z);
            m.w = __ballot_sync(FULLMASK, v1.y < T[q].w);
            *reinterpret_cast<uint4 *>(&S.msk[st][4 * q]) = m;
        }
    }
}

// LIST = true: no pair terms; every filter hit (r^2 below K.rc2_hi + margin, set to the list radius) is
// written to the neighbour list of its row atom instead.
template <bool MODE2, bool LIST>
__device__ __forceinline__ void fc_cell(FcWarp &S, const float4 *__restrict__ lpos,
                                        const int *__restrict__ cell_start, const FcGroup &G, const PairParams &P,
                                        const FcConst &K, float4 *__restrict__ frc, double &pe_tot, double &w_tot,
                                        const FcList &LO)
{
    const int lane = threadIdx.x & 31;
    const int ibeg = G.ibeg, ni = G.ni, total = G.total;
    const int cself0 = S.seg_pref[4 * (G.kk + 2) + 1];  // candidate index of the group's own atom 0
    int staged_t0 = -1;

    for (int i0 = 0; i0 < ni; i0 += 16) {
        // evaluation mapping of this pass: nrow atoms, SL slices of the mask words per atom
        const int nrow = min(16, ni - i0);
        const int SL = 32 / nrow;
        const int sl = lane / nrow, li_ = lane - sl * nrow;
        const bool myvalid = sl < SL;
        const float4 lme = lpos[ibeg + i0 + li_];
        const float zoff_me = fc_row_zoff(cell_start, G, ibeg + i0 + li_);
        const float ux = lme.x - K.h, uy = lme.y - K.h, uz = (lme.z + zoff_me) - G.hz;
        const double zme = G.hzd - (double)zoff_me;
        int rowbase = 0;                                   // list mode: entries of my atom written so far
        int qme = 0;                                       // list mode: my cell's index inside the group
        if (LIST)
            for (int k = 1; k < G.kk; k++) qme += (ibeg + i0 + li_ >= cell_start[G.cfirst + k]) ? 1 : 0;
        double tx = 0.0, ty = 0.0, tz = 0.0, pe = 0.0, w = 0.0;      // this lane's totals over the passes
        // rows of the filter for this pass (lane r < 16 prepares row r)
        __syncwarp();
        if (lane < 16) {
            const int idx = i0 + lane;
            const int slot = ibeg + min(idx, ni - 1);
            const float4 l = lpos[slot];
            const float x = l.x - K.h, y = l.y - K.h, z = (l.z + fc_row_zoff(cell_start, G, slot)) - G.hz;
            S.rax[lane] = -2.f * x;
            S.ray[lane] = -2.f * y;
            S.raz[lane] = -2.f * z;
            S.rT[lane] = (idx < ni) ? (K.rc2_hi + K.thr_margin) - fmaf(x, x, fmaf(y, y, z * z)) : -INFINITY;
        }

        for (int t0 = 0; t0 < total; t0 += FC_CAP) {
            const int cnt = min(FC_CAP, total - t0);
            const int nsteps = (cnt + 31) >> 5;
            if (t0 != staged_t0) {
                // ---- stage the candidates t0 .. t0 + cnt of the concatenated neighbour cells
                staged_t0 = t0;
                __syncwarp();
                {   // every lane labels the candidates of its two segments
                    int lo = max(G.pref0, t0) - t0, hi = min(G.pref0 + G.cnt0, t0 + cnt) - t0;
                    for (int c = lo; c < hi; c++) S.tile[c].w = __int_as_float(lane);
                    if (G.kk > 1) {
                        lo = max(G.pref1, t0) - t0, hi = min(G.pref1 + G.cnt1, t0 + cnt) - t0;
                        for (int c = lo; c < hi; c++) S.tile[c].w = __int_as_float(lane + 32);
                    }
                }
                __syncwarp();
                // four candidates per lane and batch: all loads are issued before the first store
                for (int c0 = lane; c0 < nsteps * 32; c0 += 128) {
                    float4 l[4], sg[4];
                    int kq[4];
#pragma unroll
                    for (int u = 0; u < 4; u++) {
                        const int c = c0 + 32 * u;
                        kq[u] = (c < cnt) ? __float_as_int(S.tile[c].w) : 0;
                    }
#pragma unroll
                    for (int u = 0; u < 4; u++) sg[u] = S.seg[kq[u]];
#pragma unroll
                    for (int u = 0; u < 4; u++) {
                        const int c = c0 + 32 * u;
                        l[u] = (c < cnt) ? lpos[__float_as_int(sg[u].w) + t0 + c] : make_float4(0.f, 0.f, 0.f, 0.f);
                    }
#pragma unroll
                    for (int u = 0; u < 4; u++) {
                        const int c = c0 + 32 * u;
                        float4 v;
                        v.x = l[u].x + sg[u].x;
                        v.y = l[u].y + sg[u].y;
                        v.z = l[u].z + sg[u].z;
                        v.w = fmaf(v.x, v.x, fmaf(v.y, v.y, v.z * v.z));
                        v.w = __int_as_float((__float_as_int(v.w) & ~63) | kq[u]);
                        if (c >= cnt) v = make_float4(0.f, 0.f, 0.f, INFINITY);
                        if (c < nsteps * 32) S.tile[c] = v;
                    }
                }
            }
            __syncwarp();
            if (nrow <= 4) fc_filter<1>(S, nsteps, lane);
            else if (nrow <= 8) fc_filter<2>(S, nsteps, lane);
            else if (nrow <= 12) fc_filter<3>(S, nsteps, lane);
            else fc_filter<4>(S, nsteps, lane);
            __syncwarp();
            // the pair (i, i) is not a pair
            if (lane < nrow) {
                const int cs = cself0 + i0 + lane - t0;
                if (cs >= 0 && cs < cnt) S.msk[cs >> 5][lane] &= ~(1u << (cs & 31));
            }
            __syncwarp();
            if (LIST) {
                // ---- list mode: count my hits, place my slice behind the lower slices of my atom, write
                int myhits = 0;
                if (myvalid)
                    for (int st = sl; st < nsteps; st += SL) myhits += __popc(S.msk[st][li_]);
                int before = 0, rowtot = 0;
                for (int k = 0; k < SL; k++) {
                    const int h = __shfl_sync(FULLMASK, myhits, li_ + k * nrow);
                    before += (k < sl) ? h : 0;
                    rowtot += h;
                }
                if (myvalid) {
                    const int zr = G.z0 + qme;                                  // my cell's z index
                    const bool top_me = zr == G.n - 1, below_top = ((zr == 0) ? G.n - 1 : zr - 1) == G.n - 1;
                    int pos = rowbase + before;
                    unsigned *out = LO.list + (ibeg + i0 + li_);
                    // every lane runs through its own words at its own pace (one hit per iteration)
                    int st = sl;
                    unsigned m = (st < nsteps) ? S.msk[st][li_] : 0u;
                    while (st < nsteps) {
                        if (m == 0u) {
                            st += SL;
                            if (st < nsteps) m = S.msk[st][li_];
                            continue;
                        }
                        const int b = fc_top_bit(m);
                        m ^= 1u << b;
                        const int c = st * 32 + b;
                        const int lab = __float_as_int(S.tile[c].w) & 63;
                        const int code = S.seg_code[lab];
                        const int dzr = (code >> 8) - 1 - qme;                    // candidate's cell minus mine, in z
                        const int kzc = (dzr == 0) ? 0 : (dzr > 0 ? (top_me ? 3 : 1) : (below_top ? 4 : 2));
                        const int j = __float_as_int(S.seg[lab].w) + t0 + c;
                        // cells two apart in z are farther than the list radius (cell side >= radius + 1e-3):
                        // such a hit cannot occur; if it did, a self entry offset by a cell diagonal is inert
                        unsigned e = (unsigned)j | ((unsigned)((code & 255) + 25 * kzc) << 23);
                        if (dzr < -1 || dzr > 1) e = (unsigned)(ibeg + i0 + li_) | (31u << 23);
                        if (pos < LO.cap) out[(size_t)pos * LO.npad] = e;
                        pos++;
                    }
                }
                rowbase += rowtot;
                continue;
            }
            // ---- evaluation: lane = (atom li_, slice sl) walks the hit bits of its own mask words
            // st = sl, sl + SL, ..., two hits per iteration (independent chains hide the LDS and
            // MUFU latencies); an empty word costs the lane one idle iteration.
            float fx = 0.f, fy = 0.f, fz = 0.f, sA = 0.f, sB = 0.f, sR = 0.f;   // sums of s^12, s^6, (r - rc)
            int nhit = 0, ncl = 0;
            {
                // Branch-free walk: `cur` holds the unprocessed bits of the current word (candidates
                // cb .. cb + 31), `nxt` the prefetched next word of the slice, `rem` the words after it.
                const int cstride = SL * 32;
                const int nwords = (myvalid && sl < nsteps) ? (nsteps - 1 - sl) / SL + 1 : 0;   // st = sl, sl + SL, ...
                int cb = nwords ? sl * 32 : 0;
                const unsigned *mp = &S.msk[0][0] + (nwords ? sl * 16 : 0) + li_;
                int rem = nwords - 1;                                   // words after the current one
                unsigned cur = (rem >= 0) ? *mp : 0u;
                unsigned nxt = (rem >= 1) ? mp[SL * 16] : 0u;
                mp += SL * 16;
                nhit = __popc(cur);
                while (__any_sync(FULLMASK, (cur != 0u) | (rem > 0))) {
                    // an idle slot (no bit left) reads the dummy entry behind the tile: far away, finite
                    const bool v0 = cur != 0u;
                    const int b0 = fc_top_bit(cur);
                    const int c0 = v0 ? cb + b0 : FC_CAP;
                    cur = v0 ? (cur ^ (1u << b0)) : 0u;
                    const bool v1 = cur != 0u;
                    const int b1 = fc_top_bit(cur);
                    const int c1 = v1 ? cb + b1 : FC_CAP;
                    cur = v1 ? (cur ^ (1u << b1)) : 0u;
                    const float4 u0 = S.tile[c0], u1 = S.tile[c1];
                    // refill for the next iteration while the pair terms are in flight
                    const bool need = (cur == 0u) & (rem > 0);
                    if (need) {
                        cur = nxt;
                        cb += cstride;
                        rem--;
                        mp += SL * 16;
                        nhit += __popc(nxt);
                        nxt = (rem > 0) ? *mp : 0u;
                    }
                    const float dx0 = u0.x - ux, dy0 = u0.y - uy, dz0 = u0.z - uz;
                    const float dx1 = u1.x - ux, dy1 = u1.y - uy, dz1 = u1.z - uz;
                    const float r20 = fmaf(dx0, dx0, fmaf(dy0, dy0, dz0 * dz0));
                    const float r21 = fmaf(dx1, dx1, fmaf(dy1, dy1, dz1 * dz1));
                    // p2 <= r2 < rc2_lo: FP32 term.  Everything else the filter let through (the
                    // steep part r2 < p2, the sliver around rc^2 where FP32 could misjudge the
                    // cutoff, and false positives beyond it) is decided and evaluated in FP64.
                    const bool in0 = r20 >= K.p2 && r20 < K.rc2_lo;
                    const bool in1 = r21 >= K.p2 && r21 < K.rc2_lo;
                    const bool fast0 = in0, fast1 = in1;             // the dummy entry is never in range
                    if (v0 && !in0) S.close[min(ncl++, FC_CLOSE - 1)][lane] = (unsigned short)c0;
                    if (v1 && !in1) S.close[min(ncl++, FC_CLOSE - 1)][lane] = (unsigned short)c1;
                    const float inv0 = fc_rcp(r20), inv1 = fc_rcp(r21);
                    const float s20 = K.sig2 * inv0, s21 = K.sig2 * inv1;
                    float s60 = s20 * s20 * s20, s61 = s21 * s21 * s21;
                    s60 = fast0 ? s60 : 0.f;
                    s61 = fast1 ? s61 : 0.f;
                    float fr0 = inv0 * s60 * fmaf(K.eps48, s60, -K.eps24);
                    float fr1 = inv1 * s61 * fmaf(K.eps48, s61, -K.eps24);
                    if (MODE2) {
                        const float r0 = sqrtf(r20), r1 = sqrtf(r21);
                        fr0 -= fast0 ? P.f_rcf * inv0 * r0 : 0.f;
                        fr1 -= fast1 ? P.f_rcf * inv1 * r1 : 0.f;
                        sR += fast0 ? (r0 - P.rcf) : 0.f;
                        sR += fast1 ? (r1 - P.rcf) : 0.f;
                    }
                    fx = fmaf(-fr0, dx0, fx);
                    fy = fmaf(-fr0, dy0, fy);
                    fz = fmaf(-fr0, dz0, fz);
                    sA = fmaf(s60, s60, sA);
                    sB += s60;
                    fx = fmaf(-fr1, dx1, fx);
                    fy = fmaf(-fr1, dy1, fy);
                    fz = fmaf(-fr1, dz1, fz);
                    sA = fmaf(s61, s61, sA);
                    sB += s61;
                }
            }
            // ---- FP64 part of this pass.  Queued pairs from the exact local coordinates; a lane
            // whose queue overflowed (more than FC_CLOSE slow pairs: very rare) instead rescans its
            // mask words and takes every pair outside the FP32 window.
            double dfx = 0.0, dfy = 0.0, dfz = 0.0, dpe = 0.0, dw = 0.0;
            {
                const bool ovf = ncl > FC_CLOSE;
                const int nq = ovf ? 0 : ncl;
                const int maxq = __reduce_max_sync(FULLMASK, nq);
                for (int q = 0; q < maxq; q++)
                    if (q < nq) fc_precise(S, lpos, P, K, lme, zme, t0, (int)S.close[q][lane], dfx, dfy, dfz, dpe, dw);
                if (__any_sync(FULLMASK, ovf)) {
                    if (ovf) {
                        for (int st = sl; st < nsteps; st += SL) {
                            unsigned m = S.msk[st][li_];
                            while (m) {
                                const int b = __ffs(m) - 1;
                                m &= m - 1u;
                                const int c = st * 32 + b;
                                const float4 uj = S.tile[c];
                                const float dx = uj.x - ux, dy = uj.y - uy, dz = uj.z - uz;
                                const float r2 = fmaf(dx, dx, fmaf(dy, dy, dz * dz));
                                if (!(r2 >= K.p2 && r2 < K.rc2_lo))
                                    fc_precise(S, lpos, P, K, lme, zme, t0, c, dfx, dfy, dfz, dpe, dw);
                            }
                        }
                    }
                }
            }
            // PE = 4 eps (A - B) - n ushift [+ f_rc sum(r - rc)],  W = 24 eps (2A - B) [- f_rc sum r]
            const int nin = nhit - ncl;
            tx += dfx + (double)fx;
            ty += dfy + (double)fy;
            tz += dfz + (double)fz;
            pe += dpe + P.eps4 * ((double)sA - (double)sB) - (double)nin * P.ushift;
            w += dw + P.eps24 * (2.0 * (double)sA - (double)sB);
            if (MODE2) {
                pe += P.f_rc * (double)sR;
                w -= P.f_rc * ((double)sR + (double)nin * P.rc);
            }
        }
        if (LIST) {
            if (sl == 0) {
                if (rowbase > LO.cap) atomicMax(LO.overflow, rowbase);   // the length this list needs
                int cnt = min(rowbase, LO.cap);
                // pad to a multiple of 4 with inert entries (verlet.cu: the atom itself, displaced by a cell diagonal)
                for (; cnt & 3; cnt++) LO.list[(size_t)cnt * LO.npad + (ibeg + i0 + li_)] = (unsigned)(ibeg + i0 + li_) | (31u << 23);
                LO.count[ibeg + i0 + li_] = cnt;
            }
            continue;
        }
        // ---- reduce over the slices, store
        double ox = 0.0, oy = 0.0, oz = 0.0;               // totals of the other slices of my atom
        for (int k = 1; k < SL; k++) {
            const int src = lane + k * nrow;               // < 32 for the lanes of slice 0
            ox += __shfl_sync(FULLMASK, tx, src);
            oy += __shfl_sync(FULLMASK, ty, src);
            oz += __shfl_sync(FULLMASK, tz, src);
        }
        if (sl == 0)
            frc[ibeg + i0 + li_] = make_float4((float)(tx + ox), (float)(ty + oy), (float)(tz + oz), 0.f);
        pe_tot += pe;
        w_tot += w;
    }
}

// One warp per "row group": kk <= K.kz consecutive cells of one z-column (contiguous slots, since
// z runs fastest in the cell numbering).  kz = 1 is the paper's block-per-cell;
// kz > 1 packs sparsely filled cells into one set of filter rows.  The candidates are the
// 9 columns x (kk + 2) cells around the group, i.e. the union of its cells' 27 neighbours.
// grid = (ceil(nzu / FC_WARPS), n, n): blockIdx.z = cx, blockIdx.y = cy.
template <bool MODE2, bool LIST>
__global__ void __launch_bounds__(FC_T, FC_MINB)
k_force_cell_warp(const float4 *__restrict__ lpos, const int *__restrict__ cell_start, Grid g,
                  PairParams P, FcConst K, float4 *__restrict__ frc, double *__restrict__ part_pe,
                  double *__restrict__ part_w, FcList LO, const int *__restrict__ cond)
{
    if (LIST && cond && !*cond) return;                         // conditional launch (verlet.cu)
    __shared__ FcWarp sm[FC_WARPS];
    const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
    const int n = g.n;
    // force mode: grid = (groups per column / FC_WARPS, n, n).  List mode: a small 1-D grid loops over the
    // same block indices, so that the launch costs nothing on the steps that do not rebuild.
    const int gx = (K.nzu + FC_WARPS - 1) / FC_WARPS;
    const int nblk = LIST ? gx * n * n : 1;
    for (int blk = LIST ? (int)blockIdx.x : 0; blk < nblk; blk += LIST ? (int)gridDim.x : 1) {
    const int bx = LIST ? blk % gx : (int)blockIdx.x;
    const int cy = LIST ? (blk / gx) % n : (int)blockIdx.y;
    const int cx = LIST ? blk / (gx * n) : (int)blockIdx.z;
    const int zu = bx * FC_WARPS + wid;
    double pe = 0.0, w = 0.0;
    if (zu < K.nzu) {
        const int z0 = zu * K.kz, kk = min(K.kz, n - z0);
        const int cfirst = (cx * n + cy) * n + z0;
        const int ibeg = cell_start[cfirst], ni = cell_start[cfirst + kk] - ibeg;
        if (ni > 0) {
            FcWarp &S = sm[wid];
            const int nz2 = kk + 2, nseg = 9 * nz2;
            const float hz = 0.5f * (float)kk * g.side;              // centre of the group in its frame
            int cnt[2], start[2], incl[2];
            float4 off[2];
#pragma unroll
            for (int h = 0; h < 2; h++) {
                const int sgi = lane + 32 * h;                        // segment = (column, dz)
                cnt[h] = 0; start[h] = 0;
                off[h] = make_float4(0.f, 0.f, 0.f, 0.f);
                if ((h == 0 || nseg > 32) && sgi < nseg) {
                    const int col = sgi / nz2, dz = sgi - col * nz2 - 1;     // dz = -1 .. kk
                    const int ax = col / 3 - 1, ay = col - (col / 3) * 3 - 1;
                    int nx = cx + ax, ny = cy + ay, nz = z0 + dz;
                    nx += (nx < 0) ? n : 0; nx -= (nx >= n) ? n : 0;
                    ny += (ny < 0) ? n : 0; ny -= (ny >= n) ? n : 0;
                    nz += (nz < 0) ? n : 0; nz -= (nz >= n) ? n : 0;
                    // distance between the cell origins: exact
                    off[h].x = (ax == 0) ? 0.f : (ax > 0 ? ((cx == n - 1) ? g.last : g.side) : -((nx == n - 1) ? g.last : g.side));
                    off[h].y = (ay == 0) ? 0.f : (ay > 0 ? ((cy == n - 1) ? g.last : g.side) : -((ny == n - 1) ? g.last : g.side));
                    float oz;
                    if (dz < 0) oz = -((nz == n - 1) ? g.last : g.side);
                    else oz = (float)dz * g.side + ((dz > 0 && z0 + dz - 1 == n - 1) ? (g.last - g.side) : 0.f);
                    off[h].z = oz;
                    const int nb = (nx * n + ny) * n + nz;
                    start[h] = cell_start[nb];
                    cnt[h] = cell_start[nb + 1] - start[h];
                    if (LIST) {
                        const int kx = (ax == 0) ? 0 : (ax > 0 ? ((cx == n - 1) ? 3 : 1) : ((nx == n - 1) ? 4 : 2));
                        const int ky = (ay == 0) ? 0 : (ay > 0 ? ((cy == n - 1) ? 3 : 1) : ((ny == n - 1) ? 4 : 2));
                        S.seg_code[sgi] = (kx + 5 * ky) | ((dz + 1) << 8);
                    }
                }
            }
            int carry = 0;
#pragma unroll
            for (int h = 0; h < 2; h++) {
                int v = cnt[h];
                if (h == 0 || nseg > 32) {                           // warp-uniform
#pragma unroll
                    for (int o = 1; o < 32; o <<= 1) {
                        const int y = __shfl_up_sync(FULLMASK, v, o);
                        if (lane >= o) v += y;
                    }
                }
                incl[h] = v + carry;
                carry += (h == 0 || nseg > 32) ? __shfl_sync(FULLMASK, v, 31) : 0;
            }
            const int total = carry;
            if (lane == 31) S.tile[FC_CAP] = make_float4(1.0e4f, 1.0e4f, 1.0e4f, INFINITY);
#pragma unroll
            for (int h = 0; h < 2; h++) {
                const int sgi = lane + 32 * h;
                if (sgi < FC_NSEG) {
                    const int pref = incl[h] - cnt[h];                // segments >= nseg: total
                    S.seg_pref[sgi] = pref;
                    S.seg[sgi] = make_float4(off[h].x - K.h, off[h].y - K.h, off[h].z - hz,
                                             __int_as_float(start[h] - pref));
                }
            }
            __syncwarp();
            FcGroup G;
            G.ibeg = ibeg; G.ni = ni; G.total = total; G.kk = kk; G.cfirst = cfirst;
            G.hz = hz; G.hzd = (double)hz; G.side = g.side;
            G.pref0 = incl[0] - cnt[0]; G.cnt0 = cnt[0]; G.pref1 = incl[1] - cnt[1]; G.cnt1 = cnt[1];
            G.z0 = z0; G.n = n;
            fc_cell<MODE2, LIST>(S, lpos, cell_start, G, P, K, frc, pe, w, LO);
        }
    }
    if (LIST) { __syncwarp(); continue; }
    pe = warp_sum(pe);
    w = warp_sum(w);
    if (lane == 0) {
        const int u = (cx * n + cy) * (gx * FC_WARPS) + zu;
        part_pe[u] = 0.5 * pe;                       // every pair is visited from both ends
        part_w[u] = 0.5 * w;
    }
    }
}

// Cells per row group: option "cell_group", else chosen from the mean occupancy of the grid.
static int fc_group_cells(const md_sim *s, const Grid &g)
{
    int kz = s->cell_group;
    if (kz <= 0) {
        const double occ = (double)s->N / (double)g.ncells;
        // measured optimum (B200): one cell per warp from about 11 atoms per cell on, else about
        // 22 filter rows per group
        kz = (occ >= 11.0) ? 1 : (int)(22.0 / (occ > 0.5 ? occ : 0.5) + 0.5);
        if (kz < 2) kz = (occ >= 11.0) ? 1 : 2;
    }
    if (kz > FC_KZ_MAX) kz = FC_KZ_MAX;
    if (kz < 1 || g.n < 8) kz = 1;                  // dz * side must stay exact in FP32 (L >= 16)
    return kz;
}

int ljmd_forces_cell(md_sim *s)
{
    const Grid &g = s->grid;
    // cells per row group: fill the 16 filter rows on average (option "cell_group" overrides)
    const int kz = fc_group_cells(s, g);
    const int nzu = (g.n + kz - 1) / kz;
    const dim3 grid((nzu + FC_WARPS - 1) / FC_WARPS, g.n, g.n);
    const int64_t nunits = (int64_t)grid.x * FC_WARPS * g.n * g.n;
    if (nunits > s->part_cap) return MD_ENOMEM;
    double *ppe = s->part + (size_t)s->part_cap;
    double *pw = s->part + 2 * (size_t)s->part_cap;
    const PairParams &P = s->pp;
    FcConst K;
    K.rc2_lo = (float)(P.rc2 * (1.0 - 4e-6));
    K.rc2_hi = (float)(P.rc2 * (1.0 + 4e-6));
    // Row groups of several cells stage candidates up to 3.5 cell sides from the frame centre, where
    // atoms whose global coordinate is below 4 (8 for kz = 5) lose up to 2.4e-7 (4.8e-7) of their
    // offset to FP32 rounding; the FP64 window is widened to r^2 < 1.5 sigma^2 so that every pair
    // with |df/dr| > 5 is still evaluated from the exact coordinates.
    double p2 = P.precise_r2;
    if (kz > 1 && !s->precise_r2_user) p2 = fmax(p2, 1.5 * P.sig2);
    K.p2 = (float)fmin(p2, 3.0e38);
    K.h = 0.5f * g.side;
    K.hd = (double)K.h;
    K.kz = kz;
    K.nzu = nzu;
    // farthest staged candidate from the frame centre, per dimension
    const double reach_xy = 1.5 * (double)g.last, reach_z = (0.5 * kz + 1.0) * (double)g.last;
    // FP32 rounding of the expanded form plus the 6 mantissa bits of |u|^2 that carry the segment number
    K.thr_margin = (float)(2.0e-5 * (2.0 * reach_xy * reach_xy + reach_z * reach_z) + 1e-6 * P.rc2);
    K.sig2 = P.sig2f;
    K.eps24 = P.eps24f;
    K.eps48 = 2.0f * P.eps24f;
    FcList none;
    memset(&none, 0, sizeof(none));
    if (P.mode == 2)
        k_force_cell_warp<true, false><<<grid, FC_T, 0, s->stream>>>(s->lpos, s->cell_start, g, P, K, s->frc, ppe, pw, none, nullptr);
    else
        k_force_cell_warp<false, false><<<grid, FC_T, 0, s->stream>>>(s->lpos, s->cell_start, g, P, K, s->frc, ppe, pw, none, nullptr);
    CKL(s);
    ljmd_tick(s, TAG_FORCE);
    s->n_pe = (int)nunits;
    return MD_OK;
}

// Neighbour lists (verlet.cu) through the same staging and ballot filter: cells of s->vgrid, every pair
// inside the list radius rc + skin is written instead of evaluated.  `cond`: device flag, 0 = return at once.
int ljmd_vl_build_lists(md_sim *s, const int *cond)
{
    const Grid &g = s->vgrid;
    const int kz = fc_group_cells(s, g);
    const int nzu = (g.n + kz - 1) / kz;
    const dim3 grid((nzu + FC_WARPS - 1) / FC_WARPS, g.n, g.n);
    const double rl = s->rc + s->skin;
    FcConst K;
    memset(&K, 0, sizeof(K));
    K.rc2_hi = (float)(rl * rl);                               // the filter's radius; nothing is evaluated
    K.h = 0.5f * g.side;
    K.hd = (double)K.h;
    K.kz = kz;
    K.nzu = nzu;
    const double reach_xy = 1.5 * (double)g.last, reach_z = (0.5 * kz + 1.0) * (double)g.last;
    K.thr_margin = (float)(2.0e-5 * (2.0 * reach_xy * reach_xy + reach_z * reach_z) + 1e-6 * rl * rl);
    FcList LO;
    LO.list = s->vl_list;
    LO.count = s->vl_count;
    LO.overflow = &s->vl_ctl->overflow;
    LO.npad = s->vl_npad;
    LO.cap = s->vl_cap;
    int nblk = (int)(grid.x * grid.y * grid.z), nres = (16 / FC_WARPS) * 148 * 2;   // two resident waves of blocks
    if (nblk > nres) nblk = nres;
    k_force_cell_warp<false, true><<<nblk, FC_T, 0, s->stream>>>(s->lpos, s->cell_start, g, s->pp, K, s->frc, nullptr, nullptr, LO, cond);
    CKL(s);
    return MD_OK;
}
