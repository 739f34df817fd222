/*
 * ljmd_oracle.c -- TEST INFRASTRUCTURE, NOT PRODUCT CODE.
 *
 * Plain, slow, FP64 restatement of what arXiv 0709.3225 ("Harvesting graphics
 * power for MD simulations") computes on its hot path: the Lennard-Jones pair
 * force (Eq. 1-3), an O(N^2) force loop, a separately coded linked-cell force
 * loop (Sec. 3), velocity Verlet (Sec. 2), and the rand48 linear congruential
 * generator (Sec. 4, Eq. 5-7).  Only tests/, __graft_entry__.smoke() and
 * bench.py's cpu_baseline / --impl reference legs may load this library.  It
 * shares no code, header, table or constant with the CUDA path under
 * paper_0709_3225_b200/csrc/.
 *
 * Citations are PAPER.md:<line> (the paper text in /root/reference) and the
 * numbered readings of DESIGN.md section 3 where the paper is silent.
 *
 * Pins (tests/test_oracle_*.py, run with -m "not gpu"):
 *   lj_pair            closed forms, constants at rc = 2.5, finite differences
 *   yukawa_pair        Coulomb limit kappa = 0 by hand, U at r = 1/kappa, finite differences,
 *                      two-charge force by hand, shift modes vanish at rc
 *   forces_allpairs    fcc shell sums, dimer/trimer by hand, sum F = 0,
 *                      translation invariance, scale invariance
 *   forces_cell        agreement with forces_allpairs, paper's L = 11 example
 *   verlet_*           energy conservation, dt^2 scaling, reversibility,
 *                      momentum, survey-probe trajectory values for config 1
 *   rand48_*           glibc seed48/lrand48/mrand48/drand48, skip-ahead
 *                      constants, composition laws
 * No function here is "parity unpinned".
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>

/* ------------------------------------------------------------------ O1 --
 * Pair functions.  PAPER.md:56 (Eq. 2) full LJ force, with the 1/sigma factor
 * the printed equation lacks (reading R1):
 *     f_LJ(r) = (24 eps / sigma) [ 2 (sigma/r)^13 - (sigma/r)^7 ]
 *     U_LJ(r) = 4 eps [ (sigma/r)^12 - (sigma/r)^6 ]
 * PAPER.md:61 (Eq. 3): zero for r >= rc, strict r < rc inside.
 *   mode 0: truncated only          U = U_LJ(r),            f = f_LJ(r)
 *   mode 1: energy shifted (R2)     U = U_LJ(r) - U_LJ(rc), f = f_LJ(r)
 *   mode 2: force shifted (Eq. 3)   f = f_LJ(r) - f_LJ(rc),
 *                                   U = U_LJ(r) - U_LJ(rc) + (r - rc) f_LJ(rc)
 * Outputs: *U pair energy, *f_over_r = f(r)/r.  Returns 1 if r2 < rc^2.
 */
static double u_lj(double r2, double eps, double sigma)
{
    double s2 = sigma * sigma / r2;
    double s6 = s2 * s2 * s2;
    return 4.0 * eps * (s6 * s6 - s6);
}

static double f_lj_over_r(double r2, double eps, double sigma)
{
    double s2 = sigma * sigma / r2;
    double s6 = s2 * s2 * s2;
    return 24.0 * eps * (2.0 * s6 * s6 - s6) / r2;
}

int lj_pair(int mode, double r2, double eps, double sigma, double rc,
            double *U, double *f_over_r)
{
    double rc2 = rc * rc;
    if (!(r2 < rc2)) {
        *U = 0.0;
        *f_over_r = 0.0;
        return 0;
    }
    double u = u_lj(r2, eps, sigma);
    double fr = f_lj_over_r(r2, eps, sigma);
    if (mode == 1) {
        u -= u_lj(rc2, eps, sigma);
    } else if (mode == 2) {
        double r = sqrt(r2);
        double f_rc = f_lj_over_r(rc2, eps, sigma) * rc; /* f_LJ(rc) */
        u = u - u_lj(rc2, eps, sigma) + (r - rc) * f_rc;
        fr = fr - f_rc / r;
    }
    *U = u;
    *f_over_r = fr;
    return 1;
}

/* ----------------------------------------------------------------- O1b --
 * A second pair potential through the same loops (PAPER.md:184,
 * Outlook: "it is trivial to replace this potential by other pair-potentials, including
 * the coulombic interaction"): the screened Coulomb (Yukawa) interaction between equal
 * charges,
 *     U_Y(r) = A exp(-kappa r) / r,
 *     f_Y(r) = -dU_Y/dr = A exp(-kappa r) (1/r^2 + kappa/r),
 * which is the bare Coulomb pair A/r for kappa = 0.  Truncated at rc with the same three
 * shift modes as lj_pair (the paper treats no long-range part: PAPER.md:184-188 leaves
 * Ewald-type sums to future work).  Outputs as lj_pair.
 */
static double u_yukawa(double r, double A, double kappa)
{
    return A * exp(-kappa * r) / r;
}

static double f_yukawa(double r, double A, double kappa)
{
    return A * exp(-kappa * r) * (1.0 / (r * r) + kappa / r);
}

int yukawa_pair(int mode, double r2, double A, double kappa, double rc,
                double *U, double *f_over_r)
{
    if (!(r2 < rc * rc)) {
        *U = 0.0;
        *f_over_r = 0.0;
        return 0;
    }
    double r = sqrt(r2);
    double u = u_yukawa(r, A, kappa);
    double f = f_yukawa(r, A, kappa);
    if (mode == 1) {
        u -= u_yukawa(rc, A, kappa);
    } else if (mode == 2) {
        double f_rc = f_yukawa(rc, A, kappa);
        u = u - u_yukawa(rc, A, kappa) + (r - rc) * f_rc;
        f -= f_rc;
    }
    *U = u;
    *f_over_r = f / r;
    return 1;
}

/* Which pair potential the force loops below evaluate: 0 = Lennard-Jones (eps, sigma from
 * the call), 1 = Yukawa (A, kappa set here).  Test-harness state, default 0. */
static int g_pot_kind = 0;
static double g_pot_A = 1.0, g_pot_kappa = 1.0;

void set_potential(int kind, double A, double kappa)
{
    g_pot_kind = kind;
    g_pot_A = A;
    g_pot_kappa = kappa;
}

static int pair_term(int mode, double r2, double eps, double sigma, double rc,
                     double *U, double *f_over_r)
{
    if (g_pot_kind == 1)
        return yukawa_pair(mode, r2, g_pot_A, g_pot_kappa, rc, U, f_over_r);
    return lj_pair(mode, r2, eps, sigma, rc, U, f_over_r);
}

/* ------------------------------------------------------------------ O2 --
 * All-pairs force, PAPER.md:49-52 (Eq. 1):
 *     F_i = - sum_{j != i} f(|r_j - r_i|) (r_j - r_i)/|r_j - r_i|
 * under the minimum-image convention in a cubic periodic box [0,L)^3 (R3: the
 * paper never mentions periodicity; BASELINE.json fixes it).  Half loop i<j
 * with Newton's third law.  PE = sum_{i<j} U, W = sum_{i<j} r f(r) (R12).
 * pos, F are [N][3].
 */
void forces_allpairs(int64_t N, const double *pos, double L, double rc,
                     double eps, double sigma, int mode,
                     double *F, double *PE, double *W)
{
    double pe = 0.0, w = 0.0;
    memset(F, 0, (size_t)N * 3 * sizeof(double));
    for (int64_t i = 0; i < N; i++) {
        for (int64_t j = i + 1; j < N; j++) {
            double d[3], r2 = 0.0;
            for (int c = 0; c < 3; c++) {
                d[c] = pos[3 * j + c] - pos[3 * i + c];
                d[c] -= L * nearbyint(d[c] / L);
                r2 += d[c] * d[c];
            }
            double u, fr;
            if (pair_term(mode, r2, eps, sigma, rc, &u, &fr)) {
                for (int c = 0; c < 3; c++) {
                    F[3 * i + c] -= fr * d[c];
                    F[3 * j + c] += fr * d[c];
                }
                pe += u;
                w += fr * r2;
            }
        }
    }
    *PE = pe;
    *W = w;
}

/* ------------------------------------------------------------------ O3 --
 * Cell-list force, coded separately from O2 on purpose.  PAPER.md:98 (cells of
 * side >= interaction range), :108 (one linked list per cell), :134
 * (n_x = int[L_x / rc], actual side L_x / n_x), :130 (at least 3 cells per
 * dimension).  Full shell, i-centred: every atom i visits the 27 periodic
 * neighbour cells and accumulates only F_i, U/2 and W/2.
 * Returns 0, or -1 if ncell < 3.
 */
int cell_grid(double L, double rc, int *ncell, double *side)
{
    int n = (int)floor(L / rc);
    *ncell = n;
    *side = (n > 0) ? L / n : 0.0;
    return (n >= 3) ? 0 : -1;
}

int forces_cell(int64_t N, const double *pos, double L, double rc,
                double eps, double sigma, int mode,
                double *F, double *PE, double *W)
{
    int nc;
    double side;
    if (cell_grid(L, rc, &nc, &side) != 0)
        return -1;
    int64_t ncells = (int64_t)nc * nc * nc;
    int64_t *head = (int64_t *)malloc((size_t)ncells * sizeof(int64_t));
    int64_t *next = (int64_t *)malloc((size_t)N * sizeof(int64_t));
    int *cxyz = (int *)malloc((size_t)N * 3 * sizeof(int));
    for (int64_t c = 0; c < ncells; c++)
        head[c] = -1;
    for (int64_t i = 0; i < N; i++) {
        int c[3];
        for (int k = 0; k < 3; k++) {
            c[k] = (int)floor(pos[3 * i + k] / side);
            if (c[k] > nc - 1) c[k] = nc - 1;   /* R14: clamp */
            if (c[k] < 0) c[k] = 0;
            cxyz[3 * i + k] = c[k];
        }
        int64_t id = ((int64_t)c[0] * nc + c[1]) * nc + c[2];
        next[i] = head[id];
        head[id] = i;
    }
    /* per-atom halves of U and W, summed in atom order after the loop: the result does not
     * depend on the number of threads */
    double *pei = (double *)malloc((size_t)N * sizeof(double));
    double *wi = (double *)malloc((size_t)N * sizeof(double));
#pragma omp parallel for schedule(static)
    for (int64_t i = 0; i < N; i++) {
        double fi[3] = {0.0, 0.0, 0.0};
        double pe = 0.0, w = 0.0;
        for (int ax = -1; ax <= 1; ax++)
        for (int ay = -1; ay <= 1; ay++)
        for (int az = -1; az <= 1; az++) {
            int bx = (cxyz[3 * i + 0] + ax + nc) % nc;
            int by = (cxyz[3 * i + 1] + ay + nc) % nc;
            int bz = (cxyz[3 * i + 2] + az + nc) % nc;
            int64_t id = ((int64_t)bx * nc + by) * nc + bz;
            for (int64_t j = head[id]; j >= 0; j = next[j]) {
                if (j == i) continue;
                double d[3], r2 = 0.0;
                for (int c = 0; c < 3; c++) {
                    d[c] = pos[3 * j + c] - pos[3 * i + c];
                    d[c] -= L * nearbyint(d[c] / L);
                    r2 += d[c] * d[c];
                }
                double u, fr;
                if (pair_term(mode, r2, eps, sigma, rc, &u, &fr)) {
                    for (int c = 0; c < 3; c++)
                        fi[c] -= fr * d[c];
                    pe += 0.5 * u;
                    w += 0.5 * fr * r2;
                }
            }
        }
        for (int c = 0; c < 3; c++)
            F[3 * i + c] = fi[c];
        pei[i] = pe;
        wi[i] = w;
    }
    double pe = 0.0, w = 0.0;
    for (int64_t i = 0; i < N; i++) {
        pe += pei[i];
        w += wi[i];
    }
    *PE = pe;
    *W = w;
    free(pei);
    free(wi);
    free(head);
    free(next);
    free(cxyz);
    return 0;
}

/* Pairs whose classification at the cutoff is numerically ambiguous for an
 * FP32 evaluator (R16): ordered pairs (i,j), i != j, with
 * |r^2/rc^2 - 1| < tol.  Writes up to cap pairs as (i,j) into out; returns the
 * total count found.  O(N^2): for small N only; forces_cell-sized systems use
 * near_cutoff_pairs_cell.
 */
int64_t near_cutoff_pairs(int64_t N, const double *pos, double L, double rc,
                          double tol, int64_t *out, int64_t cap)
{
    int64_t n = 0;
    double rc2 = rc * rc;
    for (int64_t i = 0; i < N; i++)
        for (int64_t j = 0; j < N; j++) {
            if (i == j) continue;
            double r2 = 0.0;
            for (int c = 0; c < 3; c++) {
                double d = pos[3 * j + c] - pos[3 * i + c];
                d -= L * nearbyint(d / L);
                r2 += d * d;
            }
            if (fabs(r2 / rc2 - 1.0) < tol) {
                if (n < cap) {
                    out[2 * n] = i;
                    out[2 * n + 1] = j;
                }
                n++;
            }
        }
    return n;
}

/* The same list through the linked cells of forces_cell (27 periodic neighbour
 * cells of every atom), for systems where the O(N^2) loop above takes hours.
 * Needs rc (1 + tol) <= cell side, i.e. tol small; returns -1 if ncell < 3.
 * Pairs come out ordered by i (then by cell walk order), serial loop.
 */
int64_t near_cutoff_pairs_cell(int64_t N, const double *pos, double L, double rc,
                               double tol, int64_t *out, int64_t cap)
{
    int nc;
    double side;
    if (cell_grid(L, rc, &nc, &side) != 0)
        return -1;
    int64_t ncells = (int64_t)nc * nc * nc;
    int64_t *head = (int64_t *)malloc((size_t)ncells * sizeof(int64_t));
    int64_t *next = (int64_t *)malloc((size_t)N * sizeof(int64_t));
    int *cxyz = (int *)malloc((size_t)N * 3 * sizeof(int));
    for (int64_t c = 0; c < ncells; c++)
        head[c] = -1;
    for (int64_t i = 0; i < N; i++) {
        int c[3];
        for (int k = 0; k < 3; k++) {
            c[k] = (int)floor(pos[3 * i + k] / side);
            if (c[k] > nc - 1) c[k] = nc - 1;
            if (c[k] < 0) c[k] = 0;
            cxyz[3 * i + k] = c[k];
        }
        int64_t id = ((int64_t)c[0] * nc + c[1]) * nc + c[2];
        next[i] = head[id];
        head[id] = i;
    }
    int64_t n = 0;
    double rc2 = rc * rc;
    for (int64_t i = 0; i < N; i++)
        for (int ax = -1; ax <= 1; ax++)
        for (int ay = -1; ay <= 1; ay++)
        for (int az = -1; az <= 1; az++) {
            int bx = (cxyz[3 * i + 0] + ax + nc) % nc;
            int by = (cxyz[3 * i + 1] + ay + nc) % nc;
            int bz = (cxyz[3 * i + 2] + az + nc) % nc;
            int64_t id = ((int64_t)bx * nc + by) * nc + bz;
            for (int64_t j = head[id]; j >= 0; j = next[j]) {
                if (j == i) continue;
                double r2 = 0.0;
                for (int c = 0; c < 3; c++) {
                    double d = pos[3 * j + c] - pos[3 * i + c];
                    d -= L * nearbyint(d / L);
                    r2 += d * d;
                }
                if (fabs(r2 / rc2 - 1.0) < tol) {
                    if (n < cap) {
                        out[2 * n] = i;
                        out[2 * n + 1] = j;
                    }
                    n++;
                }
            }
        }
    free(head);
    free(next);
    free(cxyz);
    return n;
}

/* ------------------------------------------------------------------ O4 --
 * Velocity Verlet, PAPER.md:64 ("The Velocity Verlet algorithm was applied",
 * ref. [19]); step order from BASELINE.json north_star (R4): half-kick, drift
 * with periodic wrap, force evaluation, half-kick.  Mass = 1.
 *     v += (dt/2) F;  x += dt v;  x -= L floor(x/L) (x == L -> 0, R14);
 *     F, PE, W <- forces(x);  v += (dt/2) F;  KE = (1/2) sum v^2.
 * algo 0 = forces_allpairs, 1 = forces_cell.  F must hold the forces at the
 * current positions on entry (call verlet_forces first).
 */
int verlet_forces(int64_t N, const double *pos, double L, double rc,
                  double eps, double sigma, int mode, int algo,
                  double *F, double *PE, double *W)
{
    if (algo == 0) {
        forces_allpairs(N, pos, L, rc, eps, sigma, mode, F, PE, W);
        return 0;
    }
    return forces_cell(N, pos, L, rc, eps, sigma, mode, F, PE, W);
}

double kinetic_energy(int64_t N, const double *vel)
{
    double ke = 0.0;
    for (int64_t k = 0; k < 3 * N; k++)
        ke += vel[k] * vel[k];
    return 0.5 * ke;
}

int verlet_step(int64_t N, double *pos, double *vel, double *F, double L,
                double rc, double eps, double sigma, double dt, int mode,
                int algo, double *KE, double *PE, double *W)
{
    for (int64_t k = 0; k < 3 * N; k++) {
        vel[k] += 0.5 * dt * F[k];
        pos[k] += dt * vel[k];
        pos[k] -= L * floor(pos[k] / L);
        if (pos[k] >= L) pos[k] = 0.0;
    }
    int rcode = verlet_forces(N, pos, L, rc, eps, sigma, mode, algo, F, PE, W);
    if (rcode != 0) return rcode;
    for (int64_t k = 0; k < 3 * N; k++)
        vel[k] += 0.5 * dt * F[k];
    *KE = kinetic_energy(N, vel);
    return 0;
}

/* nsteps steps; trace (if not NULL) receives [nsteps+1][3] = KE, PE, W at
 * t = 0 .. nsteps.  Forces are evaluated at entry. */
int verlet_run(int64_t N, double *pos, double *vel, double *F, double L,
               double rc, double eps, double sigma, double dt, int mode,
               int algo, int64_t nsteps, double *trace)
{
    double ke, pe, w;
    int rcode = verlet_forces(N, pos, L, rc, eps, sigma, mode, algo, F, &pe, &w);
    if (rcode != 0) return rcode;
    ke = kinetic_energy(N, vel);
    if (trace) { trace[0] = ke; trace[1] = pe; trace[2] = w; }
    for (int64_t s = 1; s <= nsteps; s++) {
        rcode = verlet_step(N, pos, vel, F, L, rc, eps, sigma, dt, mode, algo,
                            &ke, &pe, &w);
        if (rcode != 0) return rcode;
        if (trace) {
            trace[3 * s] = ke; trace[3 * s + 1] = pe; trace[3 * s + 2] = w;
        }
    }
    return 0;
}

/* ------------------------------------------------------------------ O5 --
 * rand48, PAPER.md:142-146 (Eq. 5): x_{n+1} = a x_n + c mod 2^48 with
 * a = 0x5DEECE66D, c = 0xB; the output Y_{n+1} is taken from the NEW state
 * (R8) as its most-significant bits (R7).
 *   kind 0: uint32  x >> 16          (32 high bits, mrand48 bit pattern)
 *   kind 1: uint32  x >> 17          (31 high bits, lrand48)
 *   kind 2: double  x * 2^-48        (drand48, R10)
 *   kind 3: uint64  x                (raw 48-bit state)
 */
#define R48_A 0x5DEECE66DULL
#define R48_C 0xBULL
#define R48_MASK ((1ULL << 48) - 1)

uint64_t rand48_next(uint64_t x)
{
    return (R48_A * x + R48_C) & R48_MASK;
}

/* Sequential generation, stream-major: out[s*ndraws + d] is draw d of stream
 * s; seeds[s] is replaced by the state after ndraws draws (PAPER.md:160-162,
 * "the thread saves the current state"). */
void rand48_fill_seq(uint64_t *seeds, int64_t nstreams, int64_t ndraws,
                     int kind, void *out)
{
    for (int64_t s = 0; s < nstreams; s++) {
        uint64_t x = seeds[s];
        for (int64_t d = 0; d < ndraws; d++) {
            x = rand48_next(x);
            int64_t k = s * ndraws + d;
            if (kind == 0) ((uint32_t *)out)[k] = (uint32_t)(x >> 16);
            else if (kind == 1) ((uint32_t *)out)[k] = (uint32_t)(x >> 17);
            else if (kind == 2) ((double *)out)[k] = (double)x * 0x1p-48;
            else ((uint64_t *)out)[k] = x;
        }
        seeds[s] = x;
    }
}

/* Skip-ahead constants, PAPER.md:150-156 (Eq. 6-7) with the upper bound of the
 * sum corrected to m-1 (R5):  x_{n+m} = A x_n + C,  A = a^m,
 * C = sum_{i=0}^{m-1} a^i c, all mod 2^48.  Written out literally as the
 * m-term recurrence (A,C) <- (a A, a C + c); O(m), for checking only. */
void rand48_skip_consts_linear(uint64_t m, uint64_t *A, uint64_t *C)
{
    uint64_t a_m = 1, c_m = 0;
    for (uint64_t i = 0; i < m; i++) {
        a_m = (R48_A * a_m) & R48_MASK;
        c_m = (R48_A * c_m + R48_C) & R48_MASK;
    }
    *A = a_m;
    *C = c_m;
}

/* The same constants by composing affine maps, (A1,C1) o (A2,C2) =
 * (A1 A2, A1 C2 + C1), with square-and-multiply: O(log m). */
void rand48_skip_consts(uint64_t m, uint64_t *A, uint64_t *C)
{
    uint64_t ra = 1, rc = 0;            /* identity */
    uint64_t pa = R48_A, pc = R48_C;    /* one step, then squared repeatedly */
    while (m) {
        if (m & 1) {
            rc = (pa * rc + pc) & R48_MASK;
            ra = (pa * ra) & R48_MASK;
        }
        pc = (pa * pc + pc) & R48_MASK;
        pa = (pa * pa) & R48_MASK;
        m >>= 1;
    }
    *A = ra;
    *C = rc;
}

uint64_t rand48_skip(uint64_t x, uint64_t m)
{
    uint64_t A, C;
    rand48_skip_consts(m, &A, &C);
    return (A * x + C) & R48_MASK;
}

/* Leap-frog generation exactly as PAPER.md:158-162 describes it: S lanes, lane
 * i starts from x_{i+1} (generated serially from the seed) and repeatedly
 * applies x <- A_S x + C_S; outputs interleave to the sequential series.
 * ndraws need not be a multiple of S.  Raw 48-bit states out. */
void rand48_leapfrog(uint64_t seed, int64_t S, int64_t ndraws, uint64_t *out)
{
    uint64_t A, C;
    rand48_skip_consts((uint64_t)S, &A, &C);
    uint64_t *lane = (uint64_t *)malloc((size_t)S * sizeof(uint64_t));
    uint64_t x = seed;
    for (int64_t i = 0; i < S; i++) {
        x = rand48_next(x);
        lane[i] = x;
    }
    for (int64_t base = 0; base < ndraws; base += S)
        for (int64_t i = 0; i < S && base + i < ndraws; i++) {
            out[base + i] = lane[i];
            lane[i] = (A * lane[i] + C) & R48_MASK;
        }
    free(lane);
}

/* ------------------------------------------------------------------ O6 --
 * Maxwell-Boltzmann start velocities from ONE rand48 stream (SURVEY 8(d) input recipe, DESIGN.md
 * section 4; the paper names rand48 as the generator for such uses).
 * For atom i, component c, in order: u1, u2 = the next two draws x * 2^-48;
 *     v = sqrt(T) sqrt(-2 ln(1 - u1)) cos(2 pi u2);
 * then the mean over the atoms is subtracted per component and all velocities are scaled so
 * that sum v^2 = 3 N T (R11).  vel: [N][3] doubles out; *state: in the start state x0, out the
 * state after the 6 N draws.  The GPU counterpart is md_init_velocities.
 */
void mb_velocities(int64_t N, double T, uint64_t *state, double *vel)
{
    const double two_pi = 6.283185307179586476925286766559;
    uint64_t x = *state;
    double mean[3] = {0.0, 0.0, 0.0};
    for (int64_t i = 0; i < N; i++)
        for (int c = 0; c < 3; c++) {
            x = rand48_next(x);
            double u1 = (double)x * 0x1p-48;
            x = rand48_next(x);
            double u2 = (double)x * 0x1p-48;
            double v = sqrt(T) * sqrt(-2.0 * log(1.0 - u1)) * cos(two_pi * u2);
            vel[3 * i + c] = v;
            mean[c] += v;
        }
    for (int c = 0; c < 3; c++) mean[c] /= (double)N;
    double s2 = 0.0;
    for (int64_t i = 0; i < N; i++)
        for (int c = 0; c < 3; c++) {
            vel[3 * i + c] -= mean[c];
            s2 += vel[3 * i + c] * vel[3 * i + c];
        }
    double scale = sqrt(3.0 * (double)N * T / s2);
    for (int64_t k = 0; k < 3 * N; k++) vel[k] *= scale;
    *state = x;
}

/* ----------------------------------------------------------------- O6b --
 * Andersen thermostat with rand48 (the paper names thermostats among the uses of
 * its generator; the scheme itself is the textbook one of the paper's
 * ref. [19]).  Reading taken (R24): after the second half-kick of step t (t = 0, 1, ... since
 * the thermostat was switched on) every atom i collides independently with probability
 * thr / 2^32: ONE rand48 stream with start state seed48; (t, i) owns the 7 draws starting at index
 * 7 (t N + i).  Draw 0 decides: collision iff its 32 high bits (x >> 16) are < thr (an integer
 * comparison, so both sides take the same decision).  Draws 1..6 give u1, u2 per component and
 * v_c = sqrt(T) sqrt(-2 ln(1 - u1)) cos(2 pi u2); they are skipped when there is no collision.
 * vel: [N][3] doubles, updated in place.  Returns the number of collisions.
 */
int64_t andersen_collide(int64_t N, double *vel, double T, uint32_t thr, uint64_t seed48, int64_t t)
{
    const double two_pi = 6.283185307179586476925286766559;
    int64_t ncoll = 0;
    uint64_t x = seed48;
    /* sequential walk to the first draw of step t: plain and slow on purpose */
    for (int64_t k = 0; k < 7 * t * N; k++) x = rand48_next(x);
    for (int64_t i = 0; i < N; i++) {
        uint64_t d[7];
        for (int k = 0; k < 7; k++) { x = rand48_next(x); d[k] = x; }
        if ((uint32_t)(d[0] >> 16) < thr) {
            ncoll++;
            for (int c = 0; c < 3; c++) {
                double u1 = (double)d[1 + 2 * c] * 0x1p-48, u2 = (double)d[2 + 2 * c] * 0x1p-48;
                vel[3 * i + c] = sqrt(T) * sqrt(-2.0 * log(1.0 - u1)) * cos(two_pi * u2);
            }
        }
    }
    return ncoll;
}
