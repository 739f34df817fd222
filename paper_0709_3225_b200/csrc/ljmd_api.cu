// C ABI of libljmd_b200.so (include/ljmd.h): argument validation, buffer ownership, the
// stale-force state machine and the per-step kernel sequence.  No arithmetic of the method
// happens on the host: every step of the path runs in the kernels of this library.
#include <math.h>
#include <stdio.h>
#include <stdlib.h>
#include <string.h>
#include <mutex>
#include <new>
#include <unordered_map>
#include "common.cuh"

// ---- errors -------------------------------------------------------------------------
static thread_local char g_cuda_err[512] = "";

void ljmd_note_cuda_error(cudaError_t e, const char *what, const char *file, int line)
{
    snprintf(g_cuda_err, sizeof(g_cuda_err), "%s (%s) at %s:%d: %s", cudaGetErrorName(e), what, file, line,
             cudaGetErrorString(e));
}

extern "C" const char *md_last_cuda_error(void) { return g_cuda_err; }

extern "C" const char *md_strerror(int code)
{
    switch (code) {
    case MD_OK: return "MD_OK";
    case MD_EINVAL: return "MD_EINVAL: invalid argument";
    case MD_EDOMAIN: return "MD_EDOMAIN: cell list needs at least 3 cells per dimension";
    case MD_ESTATE: return "MD_ESTATE: state not set or forces stale";
    case MD_ENOMEM: return "MD_ENOMEM: allocation failed";
    case MD_ECUDA: return "MD_ECUDA: CUDA runtime error (see md_last_cuda_error)";
    case MD_EUNSUPPORTED: return "MD_EUNSUPPORTED: not implemented in this build";
    default: return "unknown md_status";
    }
}

// ---- allocator hooks ----------------------------------------------------------------
static md_alloc_fn g_alloc = nullptr;
static md_free_fn g_free = nullptr;

extern "C" int md_set_allocator(md_alloc_fn a, md_free_fn f)
{
    if ((a == nullptr) != (f == nullptr)) return MD_EINVAL;
    g_alloc = a;
    g_free = f;
    return MD_OK;
}

// Every block remembers the hook that has to release it (nullptr: cudaFree), so that the allocator may be
// changed while handles created under the previous one are still alive.
static std::mutex g_owner_mu;
static std::unordered_map<void *, md_free_fn> g_owner;

void *ljmd_dev_alloc(int64_t bytes, cudaStream_t st)
{
    if (bytes <= 0) bytes = 16;
    void *p = nullptr;
    md_free_fn owner = nullptr;
    if (g_alloc) {
        p = g_alloc(bytes, (void *)st);
        owner = g_free;
    } else {
        cudaError_t e = cudaMalloc(&p, (size_t)bytes);
        if (e != cudaSuccess) {
            ljmd_note_cuda_error(e, "cudaMalloc", __FILE__, __LINE__);
            return nullptr;
        }
    }
    if (p) {
        std::lock_guard<std::mutex> lk(g_owner_mu);
        g_owner[p] = owner;
    }
    return p;
}

void ljmd_dev_free(void *p, cudaStream_t st)
{
    if (!p) return;
    md_free_fn owner = nullptr;
    {
        std::lock_guard<std::mutex> lk(g_owner_mu);
        auto it = g_owner.find(p);
        if (it != g_owner.end()) {
            owner = it->second;
            g_owner.erase(it);
        }
    }
    if (owner) owner(p, (void *)st);
    else cudaFree(p);
}

// ---- grid and pair constants ----------------------------------------------------------
// Cells on a lattice whose spacing is a multiple of g = ulp of the binade of L, so that cell
// origins c*side are exact floats and x - origin is exact.
static void make_grid(const md_sim *s, double rc, Grid &g)
{
    double L = s->L;
    memset(&g, 0, sizeof(g));
    g.L = s->Lf;
    int e;
    frexp(L, &e);                                    // L = m 2^e, m in [0.5,1)
    double q = ldexp(1.0, e - 24);                   // ulp of floats in [2^(e-1), 2^e)
    int n = (int)floor(L / rc);
    if (n > 1023) n = 1023;                          // cell id must fit 30 bits
    double side = 0.0;
    for (; n >= 3; n--) {
        side = floor(L / n / q) * q;
        if (side >= rc) break;
    }
    if (n < 3) return;                               // g.n stays 0: cell path unavailable
    g.n = n;
    g.ncells = n * n * n;
    g.nid = g.ncells;
    g.side = (float)side;
    g.last = (float)(L - (n - 1) * side);
    g.inv_side = (float)(1.0 / side);
}

// Number of cell ids of the Morton numbering: the padded cube P^3, P the power of two >= n.
static int morton_ids(int n)
{
    int P = 1;
    while (P < n) P <<= 1;
    return P * P * P;
}

static void setup_grid(md_sim *s)
{
    s->grid_paper_n = (int)floor(s->L / s->rc);
    make_grid(s, s->rc, s->grid);
    make_grid(s, s->rc + s->skin + 1e-3, s->vgrid);  // neighbour-list path: cells wider than rc + skin (margin: see
                                                     // the list mode of force_cell.cu)
    // make_grid starts from a cleared Grid: the numbering chosen with "cell_order" is put back, so that a later
    // "skin" or "cell_skin" does not silently return the cells to the linear numbering
    if (s->cell_order && s->grid.n) {
        s->grid.morton = 1;
        s->grid.nid = morton_ids(s->grid.n);
    }
}

static void setup_pair(md_sim *s)
{
    PairParams &P = s->pp;
    double rc = s->rc, sg = s->sigma, eps = s->eps;
    P.rc = rc;
    P.rc2 = rc * rc;
    P.sig2 = sg * sg;
    P.eps24 = 24.0 * eps;
    P.eps4 = 4.0 * eps;
    double s6 = pow(sg * sg / (rc * rc), 3.0);
    P.ushift = (s->shifted >= 1) ? 4.0 * eps * (s6 * s6 - s6) : 0.0;
    P.f_rc = (s->shifted == 2) ? 24.0 * eps * (2.0 * s6 * s6 - s6) / rc : 0.0;
    P.mode = s->shifted;
    P.kind = s->pot_kind;
    P.yA = s->pot_a;
    P.ykappa = s->pot_b;
    if (!s->precise_r2_user) P.precise_r2 = 1.3 * sg * sg;       // cell path: FP64 below this r^2
    if (s->pot_kind == MD_POT_YUKAWA) {
        const double e = s->pot_a * exp(-s->pot_b * rc) / rc;       // U_Y(rc), f_Y(rc) = U_Y (1/rc + kappa)
        P.ushift = (s->shifted >= 1) ? e : 0.0;
        P.f_rc = (s->shifted == 2) ? e * (1.0 / rc + s->pot_b) : 0.0;
        P.precise_r2 = 1.0e300;         // every in-range pair in FP64: the FP32 fast branch is Lennard-Jones only
    }
    // FP32 filter threshold: rc^2 plus the worst-case rounding error of an FP32 r^2 computed
    // from box-scale coordinates (|d| error <= 2 ulp(L)), so the filter never rejects a pair
    // that is inside rc in exact arithmetic.
    double errd = 4.0 * s->L * ldexp(1.0, -23);
    double margin = 2.0 * sqrt(3.0) * (rc + errd) * errd + P.rc2 * 1e-6;
    float f = (float)(P.rc2 + margin);
    P.rc2f_filter = nextafterf(f, INFINITY);
    P.sig2f = (float)P.sig2;
    P.eps24f = (float)P.eps24;
    P.eps4f = (float)P.eps4;
    P.ushiftf = (float)P.ushift;
    P.rcf = (float)rc;
    P.f_rcf = (float)P.f_rc;
}

// ---- per-phase timing -------------------------------------------------------------------
void ljmd_tick(md_sim *s, int tag)
{
    if (!s->time_kernels) return;
    if (s->ev_n == s->ev_cap) {
        int cap = s->ev_cap ? 2 * s->ev_cap : 1024;
        cudaEvent_t *p = (cudaEvent_t *)realloc(s->ev_pool, cap * sizeof(cudaEvent_t));
        int *t = (int *)realloc(s->ev_tag, cap * sizeof(int));
        if (!p || !t) return;
        s->ev_pool = p;
        s->ev_tag = t;
        for (int k = s->ev_cap; k < cap; k++) cudaEventCreate(&s->ev_pool[k]);
        s->ev_cap = cap;
    }
    cudaEventRecord(s->ev_pool[s->ev_n], s->stream);
    s->ev_tag[s->ev_n++] = tag;
}

int ljmd_collect_ticks(md_sim *s)
{
    if (!s->time_kernels || s->ev_n == 0) return MD_OK;
    CK(cudaStreamSynchronize(s->stream));
    for (int k = 1; k < s->ev_n; k++) {
        int tag = s->ev_tag[k];
        if (tag < 0) continue;
        float ms = 0.f;
        CK(cudaEventElapsedTime(&ms, s->ev_pool[k - 1], s->ev_pool[k]));
        s->t_phase[tag] += ms;
        s->n_phase[tag]++;
    }
    s->ev_n = 0;
    return MD_OK;
}

// ---- create / destroy -----------------------------------------------------------------
// Every cached graph has buffer addresses and capacities baked into its nodes: whoever reallocates a buffer a
// captured kernel uses (ljmd_vl_grow) or changes what the kernels are launched with calls this.
void ljmd_drop_graphs(md_sim *s)
{
    for (int k = 0; k < MD_NGRAPH; k++) {
        if (s->graphs[k].exec) cudaGraphExecDestroy(s->graphs[k].exec);
        memset(&s->graphs[k], 0, sizeof(GraphEntry));
    }
}

static void free_all(md_sim *s)
{
    cudaStream_t st = s->stream;
    for (int k = 0; k < MD_NGRAPH; k++)
        if (s->graphs[k].exec) cudaGraphExecDestroy(s->graphs[k].exec);
    if (s->cap_stream) cudaStreamDestroy(s->cap_stream);
    for (int k = 0; k < s->ev_cap; k++) cudaEventDestroy(s->ev_pool[k]);
    free(s->ev_pool);
    free(s->ev_tag);
    void *ptrs[] = {s->pos, s->vel, s->frc, s->pos2, s->vel2, s->lpos, s->lpos2, s->cell_of, s->rank, s->cell_count,
                    s->cell_start, s->max_occ, s->scan_ctl, s->scan_state, s->lpos_det, s->ap_tile_done, s->vl_list, s->vl_count, s->vl_lbuild, s->vl_ctl, s->fpart, s->part, s->energies, s->xfer, s->tile_count, s->nbr_count, s->nbr_list, s->and_t_dev,
                    s->tile_start};
    for (void *p : ptrs) ljmd_dev_free(p, st);
}

extern "C" int md_create(md_sim **out, int64_t N, double L, double rc, double eps, double sigma, double dt,
                         int shifted)
{
    if (!out) return MD_EINVAL;
    *out = nullptr;
    if (N <= 0 || N > (1LL << 30) || !(L > 0) || !(rc > 0) || !(eps >= 0) || !(sigma > 0) || !(dt > 0) ||
        shifted < 0 || shifted > 2 || !isfinite(L) || !isfinite(rc) || !isfinite(eps) || !isfinite(sigma) ||
        !isfinite(dt))
        return MD_EINVAL;
    double Lr = (double)(float)L;                                   // R13
    if (rc > 0.5 * Lr) return MD_EINVAL;
    int dev;
    CK(cudaGetDevice(&dev));
    md_sim *s = new (std::nothrow) md_sim;
    if (!s) return MD_ENOMEM;
    memset(s, 0, sizeof(*s));
    s->N = N;
    s->L = Lr;
    s->rc = rc;
    s->eps = eps;
    s->sigma = sigma;
    s->dt = dt;
    s->shifted = shifted;
    s->Lf = (float)L;
    s->dtf = (float)dt;
    s->hdtf = (float)(0.5 * dt);
    s->use_graph = true;
    s->sort_every = 10;
    s->skin = 0.3 * sigma;
    s->cell_kernel = 2;
    s->vl_fuse = true;
    setup_grid(s);
    setup_pair(s);

    const int AP_T = 128;
    int niblk = (int)((N + AP_T - 1) / AP_T);
    int nsplit = (592 + niblk - 1) / niblk;
    // j chunks are multiples of 32 atoms, whatever the number of i blocks: a small system (below
    // N ~ 4000 the launch overhead rivals the computation) still spreads over many SMs, N = 500 over 64 blocks
    if (nsplit > (int)((N + 31) / 32)) nsplit = (int)((N + 31) / 32);
    if (nsplit > 64) nsplit = 64;
    if (nsplit < 1) nsplit = 1;
    s->ap_nsplit = nsplit;
    ljmd_ap_plan(s);
    int cap_ap = niblk * nsplit;
    if ((int)((N + 7) / 8) > cap_ap) cap_ap = (int)((N + 7) / 8);       // k_allpairs_eval: 8 atoms per block
    int cap_it = (int)((N + 255) / 256);
    s->part_cap = (cap_ap > cap_it ? cap_ap : cap_it) + 64;
    if (s->grid.n) {                                                   // one partial per row group (warp)
        int64_t nu = (int64_t)s->grid.n * s->grid.n * (s->grid.n + 3) + 64;
        if (nu > s->part_cap) s->part_cap = (int)nu;
    }

    cudaStream_t st = s->stream;
    size_t f4 = (size_t)N * sizeof(float4);
    s->pos = (float4 *)ljmd_dev_alloc(f4, st);
    s->vel = (float4 *)ljmd_dev_alloc(f4, st);
    s->frc = (float4 *)ljmd_dev_alloc(f4, st);
    s->pos2 = (float4 *)ljmd_dev_alloc(f4, st);
    s->vel2 = (float4 *)ljmd_dev_alloc(f4, st);
    s->lpos = (float4 *)ljmd_dev_alloc(f4, st);
    s->cell_of = (int *)ljmd_dev_alloc(N * sizeof(int), st);
    s->rank = (int *)ljmd_dev_alloc(N * sizeof(int), st);
    // n^3 cells; the padded cube of the Morton numbering is allocated when "cell_order" asks for it
    int ncells = s->grid.n ? s->grid.ncells : 1;
    s->cell_cap = ncells;
    s->cell_count = (int *)ljmd_dev_alloc((size_t)ncells * sizeof(int), st);
    s->cell_start = (int *)ljmd_dev_alloc(((size_t)ncells + 1) * sizeof(int), st);
    s->max_occ = (unsigned long long *)ljmd_dev_alloc(sizeof(unsigned long long), st);
    {
        int nscan = ncells > s->ap_sort_bins ? ncells : s->ap_sort_bins;
        s->scan_cap = nscan / 2048 + 2;
    }
    s->scan_ctl = (ScanCtl *)ljmd_dev_alloc(sizeof(ScanCtl), st);
    s->scan_state = (unsigned long long *)ljmd_dev_alloc((size_t)s->scan_cap * sizeof(unsigned long long), st);
    s->fpart = (double *)ljmd_dev_alloc((size_t)nsplit * 3 * N * sizeof(double), st);
    s->ap_tile_done = (unsigned *)ljmd_dev_alloc((size_t)niblk * sizeof(unsigned), st);
    s->part = (double *)ljmd_dev_alloc((size_t)3 * s->part_cap * sizeof(double), st);
    s->energies = (double *)ljmd_dev_alloc(3 * sizeof(double), st);
    s->and_t_dev = (uint64_t *)ljmd_dev_alloc(sizeof(uint64_t), st);
    s->xfer = (float *)ljmd_dev_alloc((size_t)N * 3 * sizeof(float), st);
    int ntiles = s->ap_sort_bins > 0 ? s->ap_sort_bins : 1;
    s->tile_count = (int *)ljmd_dev_alloc((size_t)ntiles * sizeof(int), st);
    s->tile_start = (int *)ljmd_dev_alloc(((size_t)ntiles + 1) * sizeof(int), st);
    if (!s->tile_count || !s->tile_start || !s->pos || !s->vel || !s->frc || !s->pos2 || !s->vel2 || !s->lpos || !s->cell_of || !s->rank ||
        !s->cell_count || !s->cell_start || !s->max_occ || !s->scan_ctl || !s->scan_state || !s->fpart || !s->ap_tile_done || !s->part || !s->energies || !s->xfer || !s->and_t_dev) {
        free_all(s);
        delete s;
        return MD_ENOMEM;
    }
    cudaError_t e = cudaMemsetAsync(s->cell_count, 0, (size_t)ncells * sizeof(int), st);
    if (e == cudaSuccess) e = cudaMemsetAsync(s->ap_tile_done, 0, (size_t)niblk * sizeof(unsigned), st);
    if (e == cudaSuccess) e = cudaMemsetAsync(s->max_occ, 0, sizeof(unsigned long long), st);
    if (e == cudaSuccess) {
        ScanCtl c0;
        memset(&c0, 0, sizeof(c0));
        c0.epoch = 1;                                               // 0 marks never-written look-back words
        e = cudaMemcpyAsync(s->scan_ctl, &c0, sizeof(c0), cudaMemcpyHostToDevice, st);
        if (e == cudaSuccess) e = cudaStreamSynchronize(st);         // c0 is on the stack
    }
    if (e == cudaSuccess) e = cudaMemsetAsync(s->scan_state, 0, (size_t)s->scan_cap * sizeof(unsigned long long), st);
    if (e == cudaSuccess) e = cudaMemsetAsync(s->tile_count, 0, (size_t)ntiles * sizeof(int), st);
    if (e == cudaSuccess) e = cudaMemsetAsync(s->frc, 0, f4, st);
    if (e == cudaSuccess) e = cudaMemsetAsync(s->and_t_dev, 0, sizeof(uint64_t), st);
    if (e == cudaSuccess) e = cudaStreamSynchronize(st);
    if (e != cudaSuccess) {
        ljmd_note_cuda_error(e, "md_create init", __FILE__, __LINE__);
        free_all(s);
        delete s;
        return MD_ECUDA;
    }
    *out = s;
    return MD_OK;
}

extern "C" int md_destroy(md_sim *s)
{
    if (!s) return MD_OK;
    cudaStreamSynchronize(s->stream);
    free_all(s);
    delete s;
    return MD_OK;
}

extern "C" int md_set_potential(md_sim *s, int kind, double a, double b)
{
    if (!s) return MD_EINVAL;
    if (kind != MD_POT_LJ && kind != MD_POT_YUKAWA) return MD_EINVAL;
    if (kind == MD_POT_YUKAWA && (!isfinite(a) || !isfinite(b) || b < 0.0)) return MD_EINVAL;
    CK(cudaStreamSynchronize(s->stream));
    const bool was_yukawa = s->pot_kind == MD_POT_YUKAWA;
    s->pot_kind = kind;
    s->pot_a = a;
    s->pot_b = b;
    if (kind == MD_POT_YUKAWA) s->precise_r2_user = true;          // the window stays as set below
    else if (was_yukawa) s->precise_r2_user = false;
    setup_pair(s);
    s->forces_valid = false;
    ljmd_drop_graphs(s);
    return MD_OK;
}

extern "C" int md_set_stream(md_sim *s, void *stream)
{
    if (!s) return MD_EINVAL;
    CK(cudaStreamSynchronize(s->stream));
    s->stream = (cudaStream_t)stream;
    ljmd_drop_graphs(s);
    return MD_OK;
}

// ---- state in / out -------------------------------------------------------------------
// Copy a caller array (host or device) of n floats into device staging, or back.
static int stage_in(md_sim *s, const float *src, float *dst, size_t n)
{
    CK(cudaMemcpyAsync(dst, src, n * sizeof(float), cudaMemcpyDefault, s->stream));
    return MD_OK;
}

extern "C" int md_set_state(md_sim *s, const float *pos, const float *vel)
{
    if (!s || !pos || !vel) return MD_EINVAL;
    size_t n3 = (size_t)s->N * 3;
    // stage positions in xfer and velocities in lpos (reused as scratch: 4N floats >= 3N)
    int r = stage_in(s, pos, s->xfer, n3);
    if (r) return r;
    r = stage_in(s, vel, (float *)s->lpos, n3);
    if (r) return r;
    r = ljmd_pack_state(s, s->xfer, (const float *)s->lpos);
    if (r) return r;
    CK(cudaStreamSynchronize(s->stream));
    s->has_state = true;
    s->binned = false;
    s->binned3 = false;
    s->fused_pending = false;
    s->forces_valid = false;
    s->layout = LAYOUT_NONE;
    return MD_OK;
}

static int read_out(md_sim *s, const float4 *src, float *out)
{
    int r = ljmd_unpack(s, src, s->xfer);
    if (r) return r;
    CK(cudaMemcpyAsync(out, s->xfer, (size_t)s->N * 3 * sizeof(float), cudaMemcpyDefault, s->stream));
    CK(cudaStreamSynchronize(s->stream));
    return MD_OK;
}

extern "C" int md_get_state(md_sim *s, float *pos, float *vel)
{
    if (!s) return MD_EINVAL;
    if (!s->has_state) return MD_ESTATE;
    int r;
    if (pos && vel) {
        // both arrays with one synchronisation: positions through xfer, velocities through the spare
        // scatter target pos2 (dead between force evaluations)
        float *stage2 = (float *)s->pos2;
        if ((r = ljmd_unpack(s, s->pos, s->xfer))) return r;
        if ((r = ljmd_unpack(s, s->vel, stage2))) return r;
        const size_t bytes = (size_t)s->N * 3 * sizeof(float);
        CK(cudaMemcpyAsync(pos, s->xfer, bytes, cudaMemcpyDefault, s->stream));
        CK(cudaMemcpyAsync(vel, stage2, bytes, cudaMemcpyDefault, s->stream));
        CK(cudaStreamSynchronize(s->stream));
        return MD_OK;
    }
    if (pos && (r = read_out(s, s->pos, pos))) return r;
    if (vel && (r = read_out(s, s->vel, vel))) return r;
    return MD_OK;
}

extern "C" int md_init_velocities(md_sim *s, double T, uint64_t seed48)
{
    if (!s || !(T > 0) || !isfinite(T) || (seed48 >> 48)) return MD_EINVAL;
    if (!s->has_state) return MD_ESTATE;                              // positions (and atom ids) first
    if (s->N < 2) return MD_EINVAL;                                   // the rescaling needs a spread
    const int nb = (int)((s->N + 255) / 256);
    const int64_t nscratch = 3 * s->N + 4 * (int64_t)nb + 4;
    double *scratch = (double *)ljmd_dev_alloc(nscratch * (int64_t)sizeof(double), s->stream);
    if (!scratch) return MD_ENOMEM;
    int r = ljmd_mb_velocities(s, T, seed48, scratch, scratch + 3 * s->N, scratch + 3 * s->N + 4 * (int64_t)nb);
    if (r == MD_OK && s->forces_valid) {                              // forces do not depend on v; KE does
        r = ljmd_ke_only(s);
        if (r == MD_OK) r = ljmd_reduce_energies(s);
    }
    cudaError_t e = cudaStreamSynchronize(s->stream);
    ljmd_dev_free(scratch, s->stream);
    if (r) return r;
    if (e != cudaSuccess) { ljmd_note_cuda_error(e, "md_init_velocities", __FILE__, __LINE__); return MD_ECUDA; }
    return MD_OK;
}

extern "C" int md_get_forces(md_sim *s, float *f)
{
    if (!s || !f) return MD_EINVAL;
    if (!s->has_state || !s->forces_valid) return MD_ESTATE;
    return read_out(s, s->frc, f);
}

extern "C" int md_get_energies(md_sim *s, double *KE, double *PE, double *W)
{
    if (!s) return MD_EINVAL;
    if (!s->has_state || !s->forces_valid) return MD_ESTATE;
    double h[3];
    CK(cudaMemcpyAsync(h, s->energies, sizeof(h), cudaMemcpyDeviceToHost, s->stream));
    CK(cudaStreamSynchronize(s->stream));
    if (KE) *KE = h[0];
    if (PE) *PE = h[1];
    if (W) *W = h[2];
    return MD_OK;
}

// ---- force evaluation and stepping ------------------------------------------------------
static int check_algo(md_sim *s, int algo)
{
    if (algo != MD_ALLPAIRS && algo != MD_CELL && algo != MD_VERLET) return MD_EINVAL;
    if (algo == MD_CELL && (s->grid_paper_n < 3 || s->grid.n < 3)) return MD_EDOMAIN;
    if (algo == MD_CELL && s->cell_skin_on && s->vgrid.n < 3) return MD_EDOMAIN;
    if (algo == MD_VERLET && s->vgrid.n < 3) return MD_EDOMAIN;
    return MD_OK;
}

// energy = false: forces only (PE and the virial of this evaluation can never be read: an interior step of md_step)
// fuse = true (dense cell kernel only): the force kernel's epilogue also integrates up to the next step's
// histogram (force_cell3.cu), and the next one_step starts at the scan
static int eval_forces(md_sim *s, int algo, bool energy = true, bool fuse = false)
{
    int r;
    if (algo == MD_VERLET) {
        if ((r = ljmd_forces_verlet(s, fuse))) return r;
    } else if (algo == MD_CELL && s->cell_skin_on) {
        if ((r = ljmd_forces_skincell(s, energy))) return r;
    } else if (algo == MD_CELL && s->cell_kernel >= 2) {
        if ((r = ljmd_cell_build3(s))) return r;
        ljmd_tick(s, TAG_BUILD);
        if ((r = (s->cell_kernel == 3) ? ljmd_forces_cell3(s, energy, fuse) : ljmd_forces_cell2(s, energy, fuse))) return r;
    } else if (algo == MD_CELL) {
        if ((r = ljmd_cell_build(s))) return r;
        ljmd_tick(s, TAG_BUILD);
        if ((r = ljmd_forces_cell(s))) return r;
    } else {
        if ((r = ljmd_forces_allpairs(s))) return r;
    }
    return MD_OK;
}

// One velocity-Verlet step: [pending half-kick +] half-kick + drift [+ histogram], forces,
// and on the last step of a call the closing half-kick + KE.
// energy: PE and the virial of this evaluation will be read.  may_fuse = false keeps the integrator out of the
// force kernel (the thermostat changes the velocities between the two half-kicks).
static int one_step(md_sim *s, int algo, int kicks, bool last, bool energy, bool may_fuse = true)
{
    int r;
    const bool skinc = algo == MD_CELL && s->cell_skin_on;        // slots are stable between re-sorts: the list path's integrator
    const bool k3 = algo == MD_CELL && s->cell_kernel >= 2 && !skinc;      // lean build, fusable force kernel
    const bool vfu = algo == MD_VERLET && s->vl_fuse && !s->vl_half;
    if (!((k3 || vfu) && s->fused_pending)) {          // else: the previous force kernel has integrated already
        if ((r = skinc ? ljmd_vl_kick_drift(s, kicks)
                 : (algo == MD_CELL) ? (k3 ? ljmd_kick_drift_bin3(s, kicks) : ljmd_kick_drift_bin(s, kicks))
                                   : (algo == MD_VERLET) ? ljmd_vl_kick_drift(s, kicks) : ljmd_kick_drift(s, kicks)))
            return r;
        ljmd_tick(s, TAG_INTEGRATE);
    }
    if ((r = eval_forces(s, algo, energy, !last && may_fuse && ((k3 && s->fuse_integrator) || vfu)))) return r;
    if (last) {
        if ((r = ljmd_kick_ke(s))) return r;
        ljmd_tick(s, TAG_INTEGRATE);
    }
    return MD_OK;
}

// One interior step of md_step (neither the first nor the last of the call).  With the Andersen thermostat the
// collisions follow every second half-kick, so nothing is folded into the next step and nothing is fused.
static int interior_step(md_sim *s, int algo)
{
    if (!s->and_thr) return one_step(s, algo, 2, false, false);
    int r = one_step(s, algo, 1, false, false, false);
    if (r) return r;
    if ((r = ljmd_kick_andersen(s))) return r;
    ljmd_tick(s, TAG_INTEGRATE);
    return MD_OK;
}

// Steps after which the host-side state repeats: the cell build swaps the pos/vel buffer roles
// every step; the all-pairs path re-sorts (and swaps) every sort_every steps.
static int graph_unit(const md_sim *s, int algo)
{
    if (algo == MD_CELL && s->cell_skin_on) return 1;
    if (algo == MD_CELL) return 2;
    if (algo == MD_VERLET) return (s->vl_fuse && !s->vl_half) ? 2 : 1;   // no buffer swaps but the fused integrator's (builds are decided and done on the device)
    if (s->ap_tiled && !s->ap_force_general) return 2 * s->sort_every;
    return 1;
}

// Replay up to `nunits` units of interior steps from a cached (or newly captured) graph.
// *done = steps advanced (0 if graphs turned out to be unusable: the caller launches directly).
static int replay_interior(md_sim *s, int algo, int unit, int64_t nunits, int64_t *done)
{
    *done = 0;
    cudaStream_t user = s->stream, run = user;
    if (user == nullptr || user == cudaStreamLegacy) {
        // the legacy default stream cannot be captured: use a blocking stream, which the legacy
        // stream orders itself against in both directions
        if (!s->cap_stream && cudaStreamCreateWithFlags(&s->cap_stream, cudaStreamDefault) != cudaSuccess) {
            cudaGetLastError();
            s->use_graph = false;
            return MD_OK;
        }
        run = s->cap_stream;
    }
    GraphEntry *g = nullptr;
    for (int i = 0; i < MD_NGRAPH; i++) {
        GraphEntry &e = s->graphs[i];
        if (e.exec && e.algo == algo && e.unit == unit && e.pos == (void *)s->pos && e.vel == (void *)s->vel &&
            e.lpos == (void *)s->lpos &&
            e.since_sort == s->ap_since_sort && e.layout == s->layout && e.stream == run)
            g = &e;
    }
    if (!g) {
        // capture one unit by running the ordinary host code on the capturing stream; the
        // host-side state it leaves equals the state it found (that is what defines the unit)
        int victim = 0;
        for (int i = 1; i < MD_NGRAPH; i++)
            if (s->graphs[i].stamp < s->graphs[victim].stamp) victim = i;
        GraphEntry e;
        memset(&e, 0, sizeof(e));
        e.algo = algo; e.unit = unit; e.pos = s->pos; e.vel = s->vel; e.lpos = s->lpos; e.since_sort = s->ap_since_sort;
        e.layout = s->layout; e.stream = run;
        const md_sim saved = *s;                        // plain data: restored if the capture fails
        const int64_t l0 = s->launches;
        s->stream = run;
        cudaGraph_t graph = nullptr;
        int r = MD_OK;
        if (cudaStreamBeginCapture(run, cudaStreamCaptureModeThreadLocal) != cudaSuccess) r = MD_ECUDA;
        if (r == MD_OK) {
            for (int q = 0; q < unit && r == MD_OK; q++) r = interior_step(s, algo);
            cudaError_t ce = cudaStreamEndCapture(run, &graph);
            if (ce != cudaSuccess || !graph) r = MD_ECUDA;
        }
        if (r == MD_OK && cudaGraphInstantiate(&e.exec, graph, 0) != cudaSuccess) r = MD_ECUDA;
        if (graph) cudaGraphDestroy(graph);
        const bool same = s->pos == saved.pos && s->vel == saved.vel && s->lpos == saved.lpos && s->ap_since_sort == saved.ap_since_sort &&
                          s->layout == saved.layout;
        e.launches = s->launches - l0;
        s->stream = user;
        s->launches = l0;
        s->and_t = saved.and_t;                          // nothing ran during the capture
        if (r != MD_OK || !same) {
            // nothing was executed during the capture: put the host state back and go on without graphs
            cudaGetLastError();
            if (e.exec) cudaGraphExecDestroy(e.exec);
            GraphEntry keep[MD_NGRAPH];
            memcpy(keep, s->graphs, sizeof(keep));
            cudaStream_t cs = s->cap_stream;
            *s = saved;
            memcpy(s->graphs, keep, sizeof(keep));
            s->cap_stream = cs;
            s->use_graph = false;
            return MD_OK;
        }
        if (s->graphs[victim].exec) cudaGraphExecDestroy(s->graphs[victim].exec);
        s->graphs[victim] = e;
        g = &s->graphs[victim];
    }
    g->stamp = ++s->graph_clock;
    for (int64_t u = 0; u < nunits; u++) {
        CK(cudaGraphLaunch(g->exec, run));
        s->launches += g->launches;
        if (s->and_thr) s->and_t += (uint64_t)unit;
    }
    s->graph_replays += nunits;
    if (algo == MD_CELL) s->binned = false;
    *done = nunits * unit;
    return MD_OK;
}

// Force evaluation outside the step loop.  On the neighbour-list path a list longer than the capacity is
// never silently truncated: the lists are reallocated for the length the build asked for and rebuilt.
static int eval_forces_checked(md_sim *s, int algo)
{
    int r;
    for (int attempt = 0;; attempt++) {
        if ((r = eval_forces(s, algo))) return r;
        if (algo != MD_VERLET) return MD_OK;
        int nb, ns, ovf;
        if ((r = ljmd_vl_stats(s, &nb, &ns, &ovf))) return r;
        if (!ovf) return MD_OK;
        s->forces_valid = false;
        if (attempt == 3) return MD_ENOMEM;
        if ((r = ljmd_vl_grow(s, ovf))) return r;
    }
}

extern "C" int md_compute_forces(md_sim *s, int algo)
{
    if (!s) return MD_EINVAL;
    if (!s->has_state) return MD_ESTATE;
    int r = check_algo(s, algo);
    if (r) return r;
    if ((r = eval_forces_checked(s, algo))) return r;
    if ((r = ljmd_ke_only(s))) return r;
    if ((r = ljmd_reduce_energies(s))) return r;
    CK(cudaStreamSynchronize(s->stream));
    s->forces_valid = true;
    s->forces_algo = algo;
    return MD_OK;
}

extern "C" int md_step(md_sim *s, int64_t nsteps, int algo)
{
    if (!s || nsteps < 0) return MD_EINVAL;
    if (!s->has_state) return MD_ESTATE;
    int r = check_algo(s, algo);
    if (r) return r;
    // the neighbour-list integrator needs the lists' local coordinates: evaluate first if another
    // path (or md_set_state) ran last
    if (!s->forces_valid || (algo == MD_VERLET && s->layout != LAYOUT_VERLET && nsteps > 0) ||
        (algo == MD_CELL && s->cell_skin_on && s->layout != LAYOUT_SKINCELL && nsteps > 0)) {
        if ((r = eval_forces_checked(s, algo))) return r;
        if ((r = ljmd_ke_only(s))) return r;
        s->forces_valid = true;
        s->forces_algo = algo;
    }
    ljmd_tick(s, TAG_START);
    // Inside one call the second half-kick of step k is folded into the first kernel of step
    // k + 1 (same F, separate FMAs: bit-identical velocities); only the last step runs the
    // half-kick + KE kernel, since intermediate kinetic energies are not observable.
    // Interior steps (all but the first and the last) are identical launch sequences and are
    // replayed from a CUDA graph, one unit of steps per replay.
    int64_t k = 0;
    const bool thermo = s->and_thr != 0;         // Andersen thermostat: see interior_step; the step index lives on the device
    while (k < nsteps) {
        if (k > 0 && k < nsteps - 1 && s->use_graph && !s->time_kernels) {
            const int unit = graph_unit(s, algo);
            if (nsteps - 1 - k >= unit) {
                int64_t done = 0;
                if ((r = replay_interior(s, algo, unit, (nsteps - 1 - k) / unit, &done))) return r;
                k += done;
                if (done) continue;
            }
        }
        if (thermo) {
            if ((r = one_step(s, algo, 1, false, k == nsteps - 1, false))) return r;
            if ((r = ljmd_kick_andersen(s))) return r;
            ljmd_tick(s, TAG_INTEGRATE);
        } else if ((r = one_step(s, algo, (k > 0) ? 2 : 1, k == nsteps - 1, k == nsteps - 1))) return r;
        k++;
    }
    if ((r = ljmd_reduce_energies(s))) return r;
    ljmd_tick(s, TAG_OTHER);
    if ((r = ljmd_collect_ticks(s))) return r;
    CK(cudaStreamSynchronize(s->stream));
    if (algo == MD_VERLET) {
        int nb, ns, ovf;
        if ((r = ljmd_vl_stats(s, &nb, &ns, &ovf))) return r;
        if (ovf) {
            // a list outgrew the capacity during the run: the trajectory since that build is not valid.  The
            // lists are enlarged for the next attempt; the caller has to set the state again.
            s->forces_valid = false;
            ljmd_vl_grow(s, ovf);
            return MD_ENOMEM;
        }
    }
    s->forces_algo = algo;
    s->steps_done += nsteps;
    return MD_OK;
}

// ---- options and statistics ---------------------------------------------------------------
extern "C" int md_set_option(md_sim *s, const char *key, double value)
{
    if (!s || !key) return MD_EINVAL;
    if (!strcmp(key, "graph")) s->use_graph = value != 0.0;
    else if (!strcmp(key, "time_kernels")) {
        s->time_kernels = value != 0.0;
        s->ev_n = 0;
        for (int k = 0; k < TAG_COUNT; k++) { s->t_phase[k] = 0.0; s->n_phase[k] = 0; }
    }
    else if (!strcmp(key, "precise_r2")) {
        if (!(value >= 0)) return MD_EINVAL;
        // the FP32 fast branch of the cell and list kernels is Lennard-Jones arithmetic: with another potential
        // the window must stay empty (md_set_potential), or in-range pairs would silently get LJ forces
        if (s->pot_kind != MD_POT_LJ) return MD_EINVAL;
        s->pp.precise_r2 = value;
        s->precise_r2_user = true;
    } else if (!strcmp(key, "ap_general")) {
        s->ap_force_general = value != 0.0;
    } else if (!strcmp(key, "ap_R")) {
        int R = (int)value;
        if (R != 1 && R != 2 && R != 4 && R != 8) return MD_EINVAL;
        ljmd_ap_set_R(s, R);
        s->layout = LAYOUT_NONE;
    } else if (!strcmp(key, "andersen_nu") || !strcmp(key, "andersen_T") || !strcmp(key, "andersen_seed")) {
        if (!strcmp(key, "andersen_nu")) {
            if (!(value >= 0) || !isfinite(value)) return MD_EINVAL;
            s->and_nu = value;
        } else if (!strcmp(key, "andersen_T")) {
            if (!(value > 0) || !isfinite(value)) return MD_EINVAL;
            s->and_T = value;
        } else {
            if (!(value >= 0) || value >= 281474976710656.0 || value != floor(value)) return MD_EINVAL;
            s->and_seed = (uint64_t)value;
        }
        // collision probability per atom and step nu dt as a 32-bit threshold; needs a temperature
        double p = s->and_nu * s->dt;
        if (p > 1.0) p = 1.0;
        double thr = floor(p * 4294967296.0);
        if (thr > 4294967295.0) thr = 4294967295.0;
        s->and_thr = (s->and_T > 0) ? (uint32_t)thr : 0u;
        s->and_t = 0;                                                 // the stream starts over
        CK(cudaMemsetAsync(s->and_t_dev, 0, sizeof(uint64_t), s->stream));
    } else if (!strcmp(key, "vl_fuse")) {
        s->vl_fuse = value != 0.0;
    } else if (!strcmp(key, "vl_half")) {
        s->vl_half = value != 0.0;
        s->layout = LAYOUT_NONE;                        // rebuild the lists in the other form
    } else if (!strcmp(key, "vl_naive_build")) {
        s->vl_naive_build = value != 0.0;
    } else if (!strcmp(key, "skin")) {
        if (!(value > 0) || s->vl_ctl) return MD_EINVAL;           // before the first use of MD_VERLET / skin cells
        s->skin = value;
        setup_grid(s);
    } else if (!strcmp(key, "cell_skin")) {
        // MD_CELL on cells of side >= rc + value, re-sorted only when an atom has strayed value / 2 (0 = off:
        // the cell list is rebuilt every step).  Shares the skin with MD_VERLET: set before either is used.
        if (!(value >= 0) || !isfinite(value)) return MD_EINVAL;
        if (value > 0 && value != s->skin) {
            if (s->vl_ctl) return MD_EINVAL;
            s->skin = value;
            setup_grid(s);
        }
        s->cell_skin_on = value > 0;
        s->layout = LAYOUT_NONE;
    } else if (!strcmp(key, "cell_group")) {
        if (value < 0 || value > 5) return MD_EINVAL;
        s->cell_group = (int)value;
    } else if (!strcmp(key, "cell_order")) {
        // 1 = cells numbered along a Morton curve (measurement; dense kernel only: it selects "cell_kernel" = 3)
        if (value != 0 && value != 1) return MD_EINVAL;
        if (value == 1 && !s->grid.n) return MD_EDOMAIN;
        if (value == 1 && morton_ids(s->grid.n) > s->cell_cap) {
            // the cell arrays were sized for n^3 ids at md_create: make room for the padded cube
            const int nid = morton_ids(s->grid.n);
            const int nscan = nid > s->ap_sort_bins ? nid : s->ap_sort_bins;
            const int scan_cap = nscan / 2048 + 2;
            CK(cudaStreamSynchronize(s->stream));
            int *cc = (int *)ljmd_dev_alloc((size_t)nid * sizeof(int), s->stream);
            int *cs = (int *)ljmd_dev_alloc(((size_t)nid + 1) * sizeof(int), s->stream);
            unsigned long long *ss = (unsigned long long *)ljmd_dev_alloc((size_t)scan_cap * sizeof(unsigned long long), s->stream);
            if (!cc || !cs || !ss) {
                ljmd_dev_free(cc, s->stream); ljmd_dev_free(cs, s->stream); ljmd_dev_free(ss, s->stream);
                return MD_ENOMEM;
            }
            ljmd_dev_free(s->cell_count, s->stream);
            ljmd_dev_free(s->cell_start, s->stream);
            ljmd_dev_free(s->scan_state, s->stream);
            s->cell_count = cc;
            s->cell_start = cs;
            s->scan_state = ss;
            s->cell_cap = nid;
            s->scan_cap = scan_cap;
            CK(cudaMemsetAsync(s->scan_state, 0, (size_t)scan_cap * sizeof(unsigned long long), s->stream));   // 0 = never written
            ljmd_drop_graphs(s);
        }
        s->cell_order = (int)value;
        s->grid.morton = (int)value;
        s->grid.nid = s->grid.morton ? morton_ids(s->grid.n) : s->grid.ncells;
        if (s->grid.morton) s->cell_kernel = 3;
        s->layout = LAYOUT_NONE;
        s->forces_valid = false;
        CK(cudaMemsetAsync(s->cell_count, 0, (size_t)s->grid.nid * sizeof(int), s->stream));
    } else if (!strcmp(key, "deterministic")) {
        if (value != 0 && value != 1) return MD_EINVAL;
        if (value == 1 && !s->lpos_det) {
            s->lpos_det = (float4 *)ljmd_dev_alloc((size_t)s->N * sizeof(float4), s->stream);
            if (!s->lpos_det) return MD_ENOMEM;
        }
        s->deterministic = value == 1;
        s->layout = LAYOUT_NONE;
        s->forces_valid = false;
    } else if (!strcmp(key, "fuse_integrator")) {
        s->fuse_integrator = value != 0.0;
    } else if (!strcmp(key, "cell_kernel")) {
        if (value != 1 && value != 2 && value != 3) return MD_EINVAL;
        if (s->grid.morton && value != 3) return MD_EINVAL;          // the Morton numbering is the dense kernel's only
        s->cell_kernel = (int)value;
    } else if (!strcmp(key, "sort_every")) {
        if (value < 1) return MD_EINVAL;
        s->sort_every = (int)value;
    } else return MD_EINVAL;
    ljmd_drop_graphs(s);
    return MD_OK;
}

extern "C" int md_get_stat(md_sim *s, const char *key, double *value)
{
    if (!s || !key || !value) return MD_EINVAL;
    if (!strcmp(key, "ncell")) *value = s->grid.n;
    else if (!strcmp(key, "side")) *value = s->grid.side;
    else if (!strcmp(key, "last_side")) *value = s->grid.last;
    else if (!strcmp(key, "kernel_launches")) *value = (double)s->launches;
    else if (!strcmp(key, "steps_done")) *value = (double)s->steps_done;
    else if (!strcmp(key, "graph_replays")) *value = (double)s->graph_replays;
    else if (!strcmp(key, "andersen_threshold")) *value = (double)s->and_thr;
    else if (!strcmp(key, "andersen_steps")) *value = (double)s->and_t;
    else if (!strcmp(key, "vl_builds") || !strcmp(key, "vl_steps") || !strcmp(key, "vl_overflow")) {
        int nb, ns, ovf, r = ljmd_vl_stats(s, &nb, &ns, &ovf);
        if (r) return r;
        *value = !strcmp(key, "vl_builds") ? nb : !strcmp(key, "vl_steps") ? ns : ovf;
    } else if (!strcmp(key, "vl_cap")) *value = s->vl_cap;
    else if (!strcmp(key, "ap_nsplit")) *value = s->ap_nsplit;
    else if (!strcmp(key, "ap_tiled")) *value = s->ap_tiled ? 1 : 0;
    else if (!strcmp(key, "ap_ntiles")) *value = s->ap_ntiles;
    else if (!strcmp(key, "ap_tsplit")) *value = s->ap_tsplit;
    else if (!strcmp(key, "ap_R")) *value = s->ap_R;
    else if (!strcmp(key, "t_integrate_ms")) *value = s->t_phase[TAG_INTEGRATE];
    else if (!strcmp(key, "t_build_ms")) *value = s->t_phase[TAG_BUILD];
    else if (!strcmp(key, "t_force_ms")) *value = s->t_phase[TAG_FORCE];
    else if (!strcmp(key, "t_other_ms")) *value = s->t_phase[TAG_OTHER];
    else if (!strcmp(key, "t_force2_ms")) *value = s->t_phase[TAG_FORCE2];
    else if (!strcmp(key, "nbr_cap")) *value = s->nbr_cap;
    else if (!strcmp(key, "cell_order")) *value = s->grid.morton;
    else if (!strcmp(key, "cell_ids")) *value = s->grid.nid;
    else if (!strcmp(key, "precise_r2")) *value = s->pp.precise_r2;
    else if (!strcmp(key, "n_force")) *value = (double)s->n_phase[TAG_FORCE];
    else if (!strcmp(key, "max_occupancy")) {
        unsigned long long h = 0;
        CK(cudaMemcpyAsync(&h, s->max_occ, sizeof(h), cudaMemcpyDeviceToHost, s->stream));
        CK(cudaStreamSynchronize(s->stream));
        *value = (double)(unsigned)(h & 0xffffffffull);
    } else return MD_EINVAL;
    return MD_OK;
}
