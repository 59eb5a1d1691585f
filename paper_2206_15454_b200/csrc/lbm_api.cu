// lbm_api.cu — host side of the C ABI declared in include/lbm.h: argument checking, workspace
// layout, kernel dispatch.  No torch types; the caller owns the device workspace and the stream.
#include "../../include/lbm.h"
#include "lbm_kernels.cuh"
#include "lbm_launch.cuh"

#include <cmath>
#include <cstdarg>
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <new>
#include <vector>

using namespace lbm;

static thread_local char g_err[512] = "";

static int fail(int code, const char *fmt, ...)
{
    va_list ap;
    va_start(ap, fmt);
    vsnprintf(g_err, sizeof(g_err), fmt, ap);
    va_end(ap);
    return code;
}

// for the other translation units of the library (lbm_static.cu): set the text of lbm_last_error()
int lbm_fail_msg(int code, const char *msg) { return fail(code, "%s", msg); }

#define CU_TRY(expr)                                                                          \
    do {                                                                                      \
        cudaError_t e__ = (expr);                                                             \
        if (e__ != cudaSuccess)                                                               \
            return fail(LBM_ECUDA, "%s failed: %s", #expr, cudaGetErrorString(e__));          \
    } while (0)

static inline size_t align_up(size_t v, size_t a) { return (v + a - 1) / a * a; }

constexpr int MAX_NCHUNK = 8;
constexpr size_t STAGING_BUDGET = (size_t)256 << 20;

// Size of the host-transfer staging area.  LBM_STAGING_BYTES (environment, read at every call)
// overrides the 256 MB default so that tests can force chunked transfers on small lattices.
static size_t staging_budget()
{
    const char *e = getenv("LBM_STAGING_BYTES");
    if (e && *e) {
        const long long v = atoll(e);
        if (v > 0) return (size_t)v;
    }
    return STAGING_BUDGET;
}

struct Layout {
    size_t pops, pops2, partial, acc, shift, cda, uprof, jref, sgs, flag, solid, solid_nb, fidx, ftab, frow, bflag, staging, total;
    int stage_planes;
};

static Layout make_layout(int nx, int ny, int nz, bool aa, bool mask)
{
    Layout L;
    const size_t N = (size_t)nx * ny * nz;
    size_t off = 0;
    L.pops = off; off = align_up(off + (size_t)Q * N * 4, 256);
    L.pops2 = off; if (!aa) off = align_up(off + (size_t)Q * N * 4, 256);
    // partials per row: x chunks of the step launch (<= MAX_NCHUNK), TMA tiles, or - geometry handles - one
    // per warp of a row (KParams::wpart)
    int pmax = (nx / TMA_BOX > MAX_NCHUNK) ? nx / TMA_BOX : MAX_NCHUNK;
    if ((nx + 31) / 32 > pmax) pmax = (nx + 31) / 32;
    L.partial = off; off = align_up(off + (size_t)ny * NSTAT * nz * pmax * 4, 256);
    L.acc = off; off = align_up(off + (size_t)ny * NSTAT * 8, 256);
    L.shift = off; off = align_up(off + (size_t)ny * 4 * 4, 256);
    L.cda = off; off = align_up(off + (size_t)ny * 4, 256);
    L.uprof = off; off = align_up(off + (size_t)ny * 4, 256);
    L.jref = off; off = align_up(off + (size_t)ny * 4, 256);
    L.sgs = off; off = align_up(off + (size_t)ny * 8, 256);
    L.flag = off; off += 256;
    L.solid = off; if (mask) off = align_up(off + (size_t)((nx + 31) / 32) * ny * nz * 4, 256);
    L.solid_nb = off; if (mask) off = align_up(off + (size_t)((nx + 31) / 32) * ny * nz * 4, 256);
    L.fidx = off; if (mask) off = align_up(off + N, 256);              // per-cell forest table index, 1 B/cell
    L.ftab = off; if (mask) off = align_up(off + 256 * 4, 256);
    L.frow = off; if (mask) off = align_up(off + (size_t)ny, 256);
    L.bflag = off; if (mask) off = align_up(off + (size_t)ny * nz * MAX_NCHUNK, 256);   // one byte per thread block
    const size_t plane = (size_t)16 * nx * ny;
    size_t planes = staging_budget() / plane;
    if (planes < 1) planes = 1;
    if (planes > (size_t)nz) planes = nz;
    L.stage_planes = (int)planes;
    L.staging = off; off = align_up(off + planes * plane, 256);
    L.total = off;
    return L;
}

struct lbm_s {
    int nx, ny, nz;
    long long N;
    double nu, Cs, Fb[3], Cd, Utop[3];
    std::vector<double> lad;
    uint32_t bc;
    int bot, top;
    bool aa, aax, drag_vector, mask, halo;   // aax: the x-balanced variant of the AA pattern (aa is set too)
    bool partial_launches;      // some launches cover only part of the planes (TY must divide ny)
    bool forest_codes;          // per-cell forest codes installed (geometry handles)
    bool sgs_rows;              // per-row SGS table installed (lbm_set_sgs_rows)
    long long nflagged;         // thread blocks of the step launch that hold geometry (rebuild_block_flags)
    bool slab_open, slab_sample; // between lbm_step_slab_begin and _end; that step samples
    int zg0, nzg;               // z slab: global plane of local plane 0, global nz
    int zlo, zhi;               // planes the step updates: [zlo, zhi)
    std::vector<double> nfluid; // fluid cells per y plane (nx*nz without a mask)
    int V, TX, TY, nchunk;
    int pchunks;                // x chunks per row in the layout of the statistics partials
    // TMA data path (lbm_tma.cuh): which step kinds use it (bit 0 AA even, 1 AA odd, 2 two-lattice
    // pull) and rows per tile; maps of the two population arrays (box 256 x 1 x 1 x 1)
    bool tma_ok;
    int tma_mode, tma_rows;
    int sweep;                  // 1: consecutive steps walk the rows in opposite directions (L2 reuse), 0: always forward
    CUtensorMap map_a, map_b;
    Layout L;
    char *ws;
    cudaStream_t stream;
    int device;                 // CUDA device ordinal of the workspace (-1 before lbm_bind)
    bool bound, inited;
    long long t;
    int stats_every;
    long long stats_phase, nsamples;
    long long launches;
    int init_kind;
    double U_ref, noise_frac;
    char variant[64];
    KParams kp;
    // CUDA graph of G consecutive steps (launch-bound small lattices)
    int graph_mode;              // 0 off, 1 on, 2 auto (small lattices only)
    cudaGraphExec_t gexec;       // nullptr = none cached
    int g_steps, g_parity, g_every;
    long long g_launches, g_samples;
    char *hpin;                  // pinned host mirror of the small tables [L.acc, L.flag + 4): one D2H copy per lbm_stats_read
    bool timing;
    std::vector<cudaEvent_t> ev; // start/stop pairs of the bracketed step-kernel launches
    size_t ev_used;
};
constexpr size_t MAX_TIMED = 4096;

// Every entry point that touches the device runs under the device that owns the workspace
// (recorded at lbm_bind), whatever device is current in the calling thread.
struct DevGuard {
    int prev = -1;
    bool switched = false;
    explicit DevGuard(const lbm_s *h)
    {
        if (h && h->device >= 0 && cudaGetDevice(&prev) == cudaSuccess && prev != h->device)
            switched = cudaSetDevice(h->device) == cudaSuccess;
    }
    ~DevGuard() { if (switched) cudaSetDevice(prev); }
};

static void graph_drop(lbm_s *h)
{
    if (h->gexec) cudaGraphExecDestroy(h->gexec);
    h->gexec = nullptr;
}

// measured on cfg5 (profiles/r02_README.md): the TMA stream-in is correct but 5-7 % slower than the
// per-thread loads on the AA odd step, so it is opt-in (lbm_set_tma / LBM_TMA)
constexpr int TMA_DEFAULT_MODE = 0;

static void set_variant(lbm_s *h)
{
    char tma[32] = "";
    if (h->tma_mode) snprintf(tma, sizeof(tma), "/tma%dx%d", h->tma_mode, h->tma_rows);
    snprintf(h->variant, sizeof(h->variant), "%s/v%d/tx%dx%d%s", h->aax ? "aax" : (h->aa ? "aa" : "pull2"), h->V,
             h->TX, h->TY, tma);
}

// The statistics partials are laid out with `pchunks` x chunks per row: the larger of the
// chunkings of the kernels in use.  When it changes the buffer is cleared (entries no kernel
// writes must read as zero in the stage-2 sum).
static bool warp_partials(const lbm_s *h)   // KParams::wpart
{
    static const int all = [] { const char *e = getenv("LBM_WPART"); return (e && *e) ? atoi(e) : 0; }();   // A-B switch
    return (h->mask || all) && (h->TX % 32) == 0;
}
static int want_pchunks(const lbm_s *h)
{
    int pc = h->nchunk;
    if (h->tma_mode && h->nx / TMA_BOX > pc) pc = h->nx / TMA_BOX;
    if (warp_partials(h)) pc = h->nchunk * (h->TX / 32);
    return pc;
}
static int set_pchunks(lbm_s *h)
{
    const int pc = want_pchunks(h);
    h->kp.wpart = warp_partials(h) ? 1 : 0;
    if (pc != h->pchunks) {
        h->pchunks = pc;
        graph_drop(h);
        if (h->bound) {
            h->kp.pchunks = pc;
            CU_TRY(cudaMemsetAsync(h->ws + h->L.partial, 0, h->L.acc - h->L.partial, h->stream));
        }
    }
    return LBM_OK;
}

static bool valid_top_bottom(uint32_t bc, int *bot, int *top)
{
    const int b = bc & 3u, t = (bc >> 2) & 3u;
    if (b > 1) return false;
    if ((b == 1) != (t == 2)) return false; // periodic-y needs both faces
    *bot = b; *top = t;
    return true;
}

static int pick_vec(int nx, long long N, uint32_t bc)
{
    const int req = (bc & LBM_VEC_MASK) >> LBM_VEC_SHIFT;
    if (req == 1 || req == 2 || req == 4) return (nx % req == 0) ? req : -1;
    if (req != 0) return -1;
    // A lattice of <= 2^17 cells gives the 148 SMs less than one 4-cell-per-thread warp per scheduler:
    // the step is then bound by the latency of one warp's ~1450 dependent instructions, not by
    // memory.  One cell per thread spreads it over four times as many warps (measured on cfg1,
    // 64x32x32: 20.8 against 15.1 GLUPS without statistics, 9.5 against 9.8 with).
    if (N <= (1ll << 17)) return 1;
    if (nx % 4 == 0) return 4;
    if (nx % 2 == 0) return 2;
    return 1;
}

// Block shape: TX threads along x (a divisor of the nx/V thread columns of a row, at most
// MAX_NCHUNK blocks per row), TY rows.  Whole warps per row segment, else a power of two below a
// warp, within `target` threads; a width that offers neither (nx = 350, 372: the paper's meshes)
// takes the longest row segment that fits a block of 256 threads - measured on 350x140x280: 175x1
// 39.4 GLUPS against 34.7 for 35x2 (fewer segment edges, better warp fill).
static bool pick_shape(int W, long long nrows, int target, int *TX, int *TY)
{
    int best = -1, best_score = -1;
    for (int d = 1; d <= W && d <= target; ++d) {
        if (W % d) continue;
        if (W / d > MAX_NCHUNK) continue;
        int score = d + ((d % 32 == 0) ? 100000 : 0) + ((d < 32 && (d & (d - 1)) == 0) ? 50000 : 0);
        if (score > best_score) { best_score = score; best = d; }
    }
    int cap = target;
    if (best_score < 50000) {              // irregular width: longest segment up to 256 threads
        for (int d = 1; d <= W && d <= MAX_THREADS; ++d)
            if (W % d == 0 && W / d <= MAX_NCHUNK) best = d;
        // one such segment per block once it fills more than a warp: a second row makes warps straddle
        // the rows and the statistics reduce wait for a larger block (measured on 372x62x124, 93
        // threads per row, statistics every step: 38.9 GLUPS with 93x1 against 35.3 with 93x2; 42.5
        // against 42.0 without statistics)
        cap = (best > 32) ? best : 192;
    }
    if (best < 0) return false;
    int ty = 1;
    for (int d = 1; d * best <= cap; ++d)
        if (nrows % d == 0) ty = d;
    *TX = best; *TY = ty;
    return true;
}

// Every lbm_* function below is declared extern "C" in include/lbm.h and keeps that linkage.

const char *lbm_last_error(void) { return g_err; }

int lbm_workspace_bytes(int nx, int ny, int nz, uint32_t bc_flags, size_t *bytes)
{
    if (!bytes) return fail(LBM_EINVAL, "bytes is NULL");
    if (nx < 1 || ny < 1 || nz < 1) return fail(LBM_EINVAL, "lattice sizes must be >= 1");
    if ((double)nx * ny * nz >= 2147483648.0) return fail(LBM_EINVAL, "nx*ny*nz must be < 2^31");
    *bytes = make_layout(nx, ny, nz, (bc_flags & (LBM_STORAGE_AA | LBM_STORAGE_AAX)) != 0,
                         (bc_flags & LBM_SOLID_MASK) != 0).total;
    return LBM_OK;
}

int lbm_create(lbm_t **out, int nx, int ny, int nz, double nu, double Cs, const double *body_force,
               double Cd, const double *lad_profile, uint32_t bc_flags)
{
    if (!out) return fail(LBM_EINVAL, "out is NULL");
    *out = nullptr;
    if (nx < 1 || ny < 1 || nz < 1) return fail(LBM_EINVAL, "lattice sizes must be >= 1 (got %d %d %d)", nx, ny, nz);
    if ((double)nx * ny * nz >= 2147483648.0) return fail(LBM_EINVAL, "nx*ny*nz must be < 2^31");
    if (!(nu > 0.0) || !std::isfinite(nu)) return fail(LBM_EINVAL, "nu must be > 0 (got %g)", nu);
    if (!(Cs >= 0.0) || !std::isfinite(Cs)) return fail(LBM_EINVAL, "Cs must be >= 0 (got %g)", Cs);
    if (!(Cd >= 0.0) || !std::isfinite(Cd)) return fail(LBM_EINVAL, "Cd must be >= 0 (got %g)", Cd);
    if (bc_flags & ~(0xFu | LBM_DRAG_VECTOR | LBM_SOLID_MASK | LBM_STORAGE_AA | LBM_STORAGE_AAX | LBM_Z_HALO | LBM_VEC_MASK))
        return fail(LBM_EINVAL, "unknown bits in bc_flags 0x%x", bc_flags);
    int bot, top;
    if (!valid_top_bottom(bc_flags, &bot, &top)) return fail(LBM_EINVAL, "unsupported boundary combination in bc_flags 0x%x", bc_flags);
    if (bc_flags & LBM_Z_HALO) {
        if (nz < 3) return fail(LBM_EINVAL, "LBM_Z_HALO needs nz >= 3 (two ghost planes + >= 1 interior)");
    }
    const int V = pick_vec(nx, (long long)nx * ny * nz, bc_flags);
    if (V < 0) return fail(LBM_EINVAL, "cells-per-thread override does not divide nx=%d", nx);
    lbm_s *h = new (std::nothrow) lbm_s();
    if (!h) return fail(LBM_ENOMEM, "host allocation failed");
    h->nx = nx; h->ny = ny; h->nz = nz; h->N = (long long)nx * ny * nz;
    h->nu = nu; h->Cs = Cs; h->Cd = Cd;
    for (int a = 0; a < 3; ++a) {
        h->Fb[a] = body_force ? body_force[a] : 0.0;
        if (!std::isfinite(h->Fb[a])) { delete h; return fail(LBM_EINVAL, "body_force[%d] is not finite", a); }
    }
    h->lad.assign(ny, 0.0);
    if (lad_profile)
        for (int j = 0; j < ny; ++j) {
            if (!(lad_profile[j] >= 0.0) || !std::isfinite(lad_profile[j])) { delete h; return fail(LBM_EINVAL, "lad_profile[%d] must be >= 0", j); }
            h->lad[j] = lad_profile[j];
        }
    h->bc = bc_flags; h->bot = bot; h->top = top;
    h->aax = (bc_flags & LBM_STORAGE_AAX) != 0;
    h->aa = h->aax || (bc_flags & LBM_STORAGE_AA) != 0;    // both are single-array schemes
    h->drag_vector = (bc_flags & LBM_DRAG_VECTOR) != 0;
    h->V = V;
    h->mask = (bc_flags & LBM_SOLID_MASK) != 0;
    h->halo = (bc_flags & LBM_Z_HALO) != 0;
    h->L = make_layout(nx, ny, nz, h->aa, h->mask);
    // Rows of a launch always start at a plane boundary.  A launch that covers only some planes
    // (a slab's interior; the chunked host transfers when the staging area holds fewer than nz
    // planes) has planes*ny rows, so TY must divide ny there; otherwise TY | ny*nz is enough.
    h->partial_launches = h->halo || h->L.stage_planes < nz;
    if (!pick_shape(nx / V, h->partial_launches ? (long long)ny : (long long)ny * nz, 128, &h->TX, &h->TY)) {
        delete h;
        return fail(LBM_EINVAL, "no block shape for nx=%d with %d cells per thread", nx, V);
    }
    h->nchunk = (nx / V) / h->TX;
    h->tma_ok = (V == 4) && (nx % TMA_BOX == 0) && !h->mask && !h->aax;
    h->tma_rows = (ny % 2 == 0) ? 2 : 1;
    h->tma_mode = 0;
    if (h->tma_ok) {
        h->tma_mode = TMA_DEFAULT_MODE;
        const char *e = getenv("LBM_TMA");          // tuning / A-B override: "mode[,rows]"
        if (e && *e) {
            int m = 0, r = 0;
            const int got = sscanf(e, "%d,%d", &m, &r);
            if (got >= 1 && m >= 0 && m <= 7) h->tma_mode = m;
            if (got >= 2 && (r == 1 || r == 2 || r == 4) && ny % r == 0) h->tma_rows = r;
        }
    }
    h->pchunks = want_pchunks(h);
    h->sweep = 1;
    {
        const char *e = getenv("LBM_SWEEP");        // A-B override: 0 = always forward
        if (e && *e) h->sweep = (atoi(e) != 0) ? 1 : 0;
    }
    h->zlo = h->halo ? 1 : 0; h->zhi = h->halo ? nz - 1 : nz;
    h->zg0 = h->halo ? -1 : 0; h->nzg = h->halo ? nz - 2 : nz;
    h->nfluid.assign(ny, (double)nx * (h->zhi - h->zlo));
    h->ws = nullptr; h->stream = nullptr; h->device = -1; h->bound = false; h->inited = false;
    h->t = 0; h->stats_every = 0; h->stats_phase = 0; h->nsamples = 0; h->launches = 0;
    h->init_kind = LBM_INIT_REST; h->U_ref = 0.0; h->noise_frac = 0.0;
    h->timing = false; h->ev_used = 0; h->hpin = nullptr;
    h->graph_mode = 2; h->gexec = nullptr; h->g_steps = 0; h->g_parity = 0; h->g_every = 0;
    h->g_launches = 0; h->g_samples = 0;
    h->Utop[0] = h->Utop[1] = h->Utop[2] = 0.0;
    h->forest_codes = false;
    h->sgs_rows = false;
    h->nflagged = 0;
    h->slab_open = false; h->slab_sample = false;
    set_variant(h);
    *out = h;
    return LBM_OK;
}

static int rebuild_block_flags(lbm_s *h);

int lbm_set_launch_shape(lbm_t *h, int tx, int ty)
{
    if (!h) return fail(LBM_EINVAL, "handle is NULL");
    DevGuard dg(h);
    const int W = h->nx / h->V;
    const long long rows = h->partial_launches ? (long long)h->ny : (long long)h->ny * h->nz;
    if (tx < 1 || ty < 1 || tx * ty > MAX_THREADS || W % tx || (W / tx) > MAX_NCHUNK || rows % ty)
        return fail(LBM_EINVAL, "launch shape %dx%d does not tile %d thread columns x %lld rows%s", tx, ty, W,
                    rows, h->partial_launches ? " (ty must divide ny: this handle launches plane ranges)" : "");
    graph_drop(h);
    h->TX = tx; h->TY = ty; h->nchunk = W / tx;
    h->kp.nchunk = h->nchunk;
    set_variant(h);
    int rc = set_pchunks(h);
    if (rc) return rc;
    return rebuild_block_flags(h);
}

static void fill_params(lbm_s *h)
{
    KParams &p = h->kp;
    memset(&p, 0, sizeof(p));
    p.src = reinterpret_cast<float *>(h->ws + h->L.pops);
    p.dst = h->aa ? p.src : reinterpret_cast<float *>(h->ws + h->L.pops2);
    p.nx = h->nx; p.ny = h->ny; p.nz = h->nz; p.nchunk = h->nchunk; p.pchunks = h->pchunks; p.N = h->N;
    p.wpart = warp_partials(h) ? 1 : 0;
    const double tau0 = 3.0 * h->nu + 0.5;              // R3
    p.tau0 = (float)tau0; p.tau0sq = (float)(tau0 * tau0);
    p.ksmag = (float)(18.0 * std::sqrt(2.0) * h->Cs * h->Cs); // R9: C_smag = Cs^2
    p.Fbx = (float)h->Fb[0]; p.Fby = (float)h->Fb[1]; p.Fbz = (float)h->Fb[2];
    p.cda = reinterpret_cast<const float *>(h->ws + h->L.cda);
    p.jref = reinterpret_cast<const float *>(h->ws + h->L.jref);
    p.sgs = h->sgs_rows ? reinterpret_cast<const float2 *>(h->ws + h->L.sgs) : nullptr;
    p.bot = h->bot; p.top = h->top; p.drag_vector = h->drag_vector ? 1 : 0;
    p.aax = h->aax ? 1 : 0;
    {
        // lid populations f_eq,i(1, U_top) - w_i (Eq. 3) of the five directions with c_y = -1
        static const int li[5] = {4, 8, 9, 16, 18};
        const double *U = h->Utop, uu = U[0] * U[0] + U[1] * U[1] + U[2] * U[2];
        for (int q = 0; q < 5; ++q) {
            const int i = li[q];
            const double cu = Lat::cx[i] * U[0] + Lat::cy[i] * U[1] + Lat::cz[i] * U[2];
            const double w = (i < 7) ? 1.0 / 18.0 : 1.0 / 36.0;
            p.lid[q] = (float)(w * (3.0 * cu + 4.5 * cu * cu - 1.5 * uu));
        }
    }
    p.solid = h->mask ? reinterpret_cast<const unsigned *>(h->ws + h->L.solid) : nullptr;
    p.solid_nb = h->mask ? reinterpret_cast<const unsigned *>(h->ws + h->L.solid_nb) : nullptr;
    p.nxw = (h->nx + 31) / 32;
    p.fidx = (h->mask && h->forest_codes) ? reinterpret_cast<const unsigned char *>(h->ws + h->L.fidx) : nullptr;
    p.ftab = h->mask ? reinterpret_cast<const float *>(h->ws + h->L.ftab) : nullptr;
    p.frow = h->mask ? reinterpret_cast<const unsigned char *>(h->ws + h->L.frow) : nullptr;
    p.bflag = h->mask ? reinterpret_cast<const unsigned char *>(h->ws + h->L.bflag) : nullptr;
    p.partial = nullptr; p.shift = nullptr;
    p.diverged = reinterpret_cast<int *>(h->ws + h->L.flag);
    p.uprof = reinterpret_cast<const float *>(h->ws + h->L.uprof);
    p.z0 = 0; p.z1 = h->nz; p.zoff = 0; p.Nio = h->N;
    p.zg0 = h->zg0; p.nzg = h->nzg;
    p.zv0 = h->zlo; p.zv1 = h->zhi;
}

// Tensor map of one population array viewed as a rank-4 fp32 tensor {x, y, z, slot} with a box of
// one 256-cell row segment.  cuTensorMapEncodeTiled is a driver entry point; it is looked up
// through the runtime so that the library does not link against libcuda.
static int make_tensor_map(lbm_s *h, void *base, CUtensorMap *out)
{
    typedef CUresult (*encode_fn)(CUtensorMap *, CUtensorMapDataType, cuuint32_t, void *, const cuuint64_t *,
                                  const cuuint64_t *, const cuuint32_t *, const cuuint32_t *, CUtensorMapInterleave,
                                  CUtensorMapSwizzle, CUtensorMapL2promotion, CUtensorMapFloatOOBfill);
    static encode_fn encode = nullptr;
    if (!encode) {
        void *fn = nullptr;
        cudaDriverEntryPointQueryResult q;
        CU_TRY(cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &fn, cudaEnableDefault, &q));
        if (q != cudaDriverEntryPointSuccess || !fn) return fail(LBM_ECUDA, "cuTensorMapEncodeTiled is not available");
        encode = reinterpret_cast<encode_fn>(fn);
    }
    const cuuint64_t dims[4] = {(cuuint64_t)h->nx, (cuuint64_t)h->ny, (cuuint64_t)h->nz, (cuuint64_t)Q};
    const cuuint64_t strides[3] = {(cuuint64_t)h->nx * 4, (cuuint64_t)h->nx * h->ny * 4, (cuuint64_t)h->N * 4};
    const cuuint32_t box[4] = {(cuuint32_t)TMA_BOX, 1, 1, 1};
    const cuuint32_t estr[4] = {1, 1, 1, 1};
    const CUresult r = encode(out, CU_TENSOR_MAP_DATA_TYPE_FLOAT32, 4, base, dims, strides, box, estr,
                              CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_NONE,
                              CU_TENSOR_MAP_L2_PROMOTION_NONE, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
    if (r != CUDA_SUCCESS) return fail(LBM_ECUDA, "cuTensorMapEncodeTiled failed with CUresult %d", (int)r);
    return LBM_OK;
}

int lbm_bind(lbm_t *h, void *dev_workspace, size_t bytes, void *cuda_stream)
{
    if (!h) return fail(LBM_EINVAL, "handle is NULL");
    if (!dev_workspace) return fail(LBM_EINVAL, "workspace is NULL");
    if (bytes < h->L.total) return fail(LBM_ENOMEM, "workspace too small: %zu < %zu bytes", bytes, h->L.total);
    if (reinterpret_cast<uintptr_t>(dev_workspace) % 256) return fail(LBM_ENOMEM, "workspace must be 256-byte aligned");
    {
        cudaPointerAttributes at;
        CU_TRY(cudaPointerGetAttributes(&at, dev_workspace));
        if (at.type != cudaMemoryTypeDevice && at.type != cudaMemoryTypeManaged)
            return fail(LBM_EINVAL, "workspace is not device memory");
        h->device = at.device;
    }
    DevGuard dg(h);
    graph_drop(h);
    h->ws = static_cast<char *>(dev_workspace);
    h->stream = static_cast<cudaStream_t>(cuda_stream);
    fill_params(h);
    if (h->tma_ok) {
        int rc = make_tensor_map(h, h->ws + h->L.pops, &h->map_a);
        if (rc == LBM_OK && !h->aa) rc = make_tensor_map(h, h->ws + h->L.pops2, &h->map_b);
        if (rc != LBM_OK) return rc;
    }
    std::vector<float> cda(h->ny);
    for (int j = 0; j < h->ny; ++j) cda[j] = (float)(h->Cd * h->lad[j]);
    CU_TRY(cudaMemcpyAsync(h->ws + h->L.cda, cda.data(), h->ny * 4, cudaMemcpyHostToDevice, h->stream));
    CU_TRY(cudaMemsetAsync(h->ws + h->L.acc, 0, (size_t)h->ny * NSTAT * 8, h->stream));
    CU_TRY(cudaMemsetAsync(h->ws + h->L.shift, 0, (size_t)h->ny * 16, h->stream));
    CU_TRY(cudaMemsetAsync(h->ws + h->L.flag, 0, 256, h->stream));
    CU_TRY(cudaMemsetAsync(h->ws + h->L.jref, 0, (size_t)h->ny * 4, h->stream));
    h->sgs_rows = false; h->kp.sgs = nullptr;
    CU_TRY(cudaMemsetAsync(h->ws + h->L.partial, 0, h->L.acc - h->L.partial, h->stream));
    if (h->mask) {
        const size_t mbytes = (size_t)((h->nx + 31) / 32) * h->ny * h->nz * 4;
        CU_TRY(cudaMemsetAsync(h->ws + h->L.solid, 0, mbytes, h->stream));
        CU_TRY(cudaMemsetAsync(h->ws + h->L.solid_nb, 0, mbytes, h->stream));
        CU_TRY(cudaMemsetAsync(h->ws + h->L.bflag, 0, (size_t)h->ny * h->nz * MAX_NCHUNK, h->stream));
        h->nflagged = 0;
        h->forest_codes = false;
        h->kp.fidx = nullptr;
    }
    CU_TRY(cudaStreamSynchronize(h->stream)); // cda is a local vector
    if (!h->hpin) CU_TRY(cudaHostAlloc(reinterpret_cast<void **>(&h->hpin), h->L.flag + 4 - h->L.acc, cudaHostAllocDefault));
    h->bound = true; h->inited = false;
    return LBM_OK;
}

// Rebuild the per-block geometry flags of the step launch (after a change of the mask, the forest
// codes or the block shape).
static int rebuild_block_flags(lbm_s *h)
{
    if (!h->mask || !h->bound) return LBM_OK;
    const long long nblocks = (long long)h->ny * h->nz / h->TY * h->nchunk;
    blockflag_kernel<<<(unsigned)((nblocks + 127) / 128), 128, 0, h->stream>>>(
        h->kp, h->TX * h->V, h->TY, reinterpret_cast<unsigned char *>(h->ws + h->L.bflag), nblocks);
    h->launches++;
    CU_TRY(cudaGetLastError());
    // how many blocks hold geometry: none (a mask that is all fluid, e.g. after the trip boxes have
    // been removed) => lbm_step launches the plain kernels, at no cost at all
    std::vector<unsigned char> flags((size_t)nblocks);
    CU_TRY(cudaMemcpyAsync(flags.data(), h->ws + h->L.bflag, (size_t)nblocks, cudaMemcpyDeviceToHost, h->stream));
    CU_TRY(cudaStreamSynchronize(h->stream));
    long long n = 0;
    for (unsigned char f : flags) n += f ? 1 : 0;
    h->nflagged = n;
    graph_drop(h);
    return LBM_OK;
}

int lbm_set_solid(lbm_t *h, const uint8_t *solid_host)
{
    if (!h) return fail(LBM_EINVAL, "handle is NULL");
    DevGuard dg(h);
    if (!h->mask) return fail(LBM_EINVAL, "handle was not created with LBM_SOLID_MASK");
    if (!h->bound) return fail(LBM_ESTATE, "lbm_set_solid before lbm_bind");
    // (z slab, single-array storage, even t: populations that cross a slab face sit in the ghost planes of
    // the rank that pushed them; the conversion below works on every local plane, ghosts included, and
    // the caller then repeats the halo exchange - lbm.h)
    const int nxw = (h->nx + 31) / 32;
    const size_t words = (size_t)nxw * h->ny * h->nz;
    std::vector<uint32_t> bits;
    try { bits.assign(words, 0u); } catch (...) { return fail(LBM_ENOMEM, "host allocation failed"); }
    h->nfluid.assign(h->ny, (double)h->nx * (h->zhi - h->zlo));
    if (solid_host)
        for (int z = 0; z < h->nz; ++z)
            for (int y = 0; y < h->ny; ++y) {
                const uint8_t *row = solid_host + ((size_t)z * h->ny + y) * h->nx;
                uint32_t *out = bits.data() + ((size_t)z * h->ny + y) * nxw;
                for (int x = 0; x < h->nx; ++x)
                    if (row[x]) {
                        out[x >> 5] |= 1u << (x & 31);
                        if (z >= h->zlo && z < h->zhi) h->nfluid[y] -= 1.0;
                    }
            }
    // the mask dilated by one cell in every direction (periodic x, z; y only where periodic):
    // bit = some cell within one step is solid.  The kernels skip the geometry work where it is 0.
    // A row is nxw words; the last one is ragged when nx % 32 != 0 (bits past nx stay 0).
    std::vector<uint32_t> nb;
    try { nb.assign(words, 0u); } catch (...) { return fail(LBM_ENOMEM, "host allocation failed"); }
    const bool yper = h->bot == BC_BOT_PERIODIC;
    const int lastb = (h->nx - 1) & 31;
    const uint32_t lastmask = (lastb == 31) ? 0xFFFFFFFFu : ((1u << (lastb + 1)) - 1u);
    for (int z = 0; z < h->nz; ++z)
        for (int y = 0; y < h->ny; ++y) {
            uint32_t *out = nb.data() + ((size_t)z * h->ny + y) * nxw;
            for (int dz = -1; dz <= 1; ++dz)
                for (int dy = -1; dy <= 1; ++dy) {
                    int yy = y + dy;
                    if (yy < 0 || yy >= h->ny) { if (!yper) continue; yy = (yy + h->ny) % h->ny; }
                    const int zz = (z + dz + h->nz) % h->nz;
                    const uint32_t *row = bits.data() + ((size_t)zz * h->ny + yy) * nxw;
                    for (int w = 0; w < nxw; ++w) {
                        const uint32_t m = row[w];
                        // the bit left of this word's bit 0 and the bit right of its last valid bit
                        const uint32_t lc = (w == 0) ? ((row[nxw - 1] >> lastb) & 1u) : (row[w - 1] >> 31);
                        const uint32_t rc = (w + 1 == nxw) ? (row[0] & 1u) : (row[w + 1] & 1u);
                        uint32_t v = m | (m << 1) | (m >> 1) | lc | (rc << ((w + 1 == nxw) ? lastb : 31));
                        if (w + 1 == nxw) v &= lastmask;
                        out[w] |= v;
                    }
                }
        }
    graph_drop(h);
    if (h->inited) {
        // run-time change: keep the flow.  The new mask waits in the staging area
        // while the populations are moved from the old geometry's representation to the new one.
        if (words * 4 > (size_t)(h->L.total - h->L.staging)) return fail(LBM_ENOMEM, "staging area too small for the mask");
        uint32_t *newm = reinterpret_cast<uint32_t *>(h->ws + h->L.staging);
        CU_TRY(cudaMemcpyAsync(newm, bits.data(), words * 4, cudaMemcpyHostToDevice, h->stream));
        KParams p = h->kp;
        float *arr = (!h->aa && (h->t & 1)) ? p.dst : p.src;            // the array holding state t
        const unsigned blocks = (unsigned)((h->N + 255) / 256);
        if (h->aax && (h->t & 1) == 0)
            mask_change_kernel<true, true><<<blocks, 256, 0, h->stream>>>(p, arr, p.solid, newm);
        else if (h->aax)
            mask_change_kernel<false, true><<<blocks, 256, 0, h->stream>>>(p, arr, p.solid, newm);
        else if (h->aa && (h->t & 1) == 0)
            mask_change_kernel<true><<<blocks, 256, 0, h->stream>>>(p, arr, p.solid, newm);
        else
            mask_change_kernel<false><<<blocks, 256, 0, h->stream>>>(p, arr, p.solid, newm);
        h->launches++;
        CU_TRY(cudaGetLastError());
        CU_TRY(cudaMemcpyAsync(h->ws + h->L.solid, newm, words * 4, cudaMemcpyDeviceToDevice, h->stream));
    } else {
        CU_TRY(cudaMemcpyAsync(h->ws + h->L.solid, bits.data(), words * 4, cudaMemcpyHostToDevice, h->stream));
    }
    CU_TRY(cudaMemcpyAsync(h->ws + h->L.solid_nb, nb.data(), words * 4, cudaMemcpyHostToDevice, h->stream));
    int rc = rebuild_block_flags(h);
    if (rc) return rc;
    CU_TRY(cudaStreamSynchronize(h->stream));
    return LBM_OK;
}

// Bit fields of a forest code (include/lbm.h): y | h << 10 | y_m (eighths of a cell) << 20.
static double forest_code_lad(uint32_t code, double a_fm)
{
    const int y = (int)(code & 1023u), hc = (int)((code >> 10) & 1023u);
    const double ym = (double)((code >> 20) & 4095u) / 8.0;
    if (hc == 0 || y >= hc) return 0.0;
    if (ym == 0.0) return a_fm;                              // constant LAD (Table II case 1)
    // Eq. 14 (L107) with Eq. 15 (L112) at the cell centre
    const double eta = (y + 0.5) / hc, eta_m = ym / hc;
    const double ratio = (1.0 - eta_m) / (1.0 - eta);
    const double n = (eta < eta_m) ? 6.0 : 0.5;
    return a_fm * std::exp(n * std::log(ratio) + n * (1.0 - ratio));
}

uint32_t lbm_forest_code(int hc, int y, double y_m)
{
    const uint32_t ym8 = (uint32_t)std::floor(y_m * 8.0 + 0.5);
    return ((uint32_t)y & 1023u) | (((uint32_t)hc & 1023u) << 10) | ((ym8 & 4095u) << 20);
}

int lbm_set_forest_codes(lbm_t *h, const uint32_t *code_host, double a_fm)
{
    if (!h) return fail(LBM_EINVAL, "handle is NULL");
    DevGuard dg(h);
    if (!h->mask) return fail(LBM_EINVAL, "per-cell forest codes need a geometry handle (LBM_SOLID_MASK)");
    if (!h->bound) return fail(LBM_ESTATE, "lbm_set_forest_codes before lbm_bind");
    if (!(a_fm >= 0.0) || !std::isfinite(a_fm)) return fail(LBM_EINVAL, "a_fm must be >= 0");
    graph_drop(h);
    if (!code_host) {
        h->forest_codes = false;
        h->kp.fidx = nullptr;
        int rc0 = rebuild_block_flags(h);
        if (rc0) return rc0;
        CU_TRY(cudaStreamSynchronize(h->stream));
        return LBM_OK;
    }
    // distinct codes -> table of C_D a_f (fp32), one byte per cell indexes it
    std::vector<uint8_t> idx;
    std::vector<uint8_t> frow(h->ny, 0);
    try { idx.assign((size_t)h->N, 0); } catch (...) { return fail(LBM_ENOMEM, "host allocation failed"); }
    std::vector<uint32_t> codes;                             // codes[k-1] has table index k
    std::vector<float> tab(256, 0.f);
    uint32_t last = 0; int last_k = 0;
    for (long long n = 0; n < h->N; ++n) {
        const uint32_t c = code_host[n];
        if (!c) continue;
        int k = 0;
        if (c == last) k = last_k;
        else {
            for (size_t q = 0; q < codes.size(); ++q) if (codes[q] == c) { k = (int)q + 1; break; }
            if (!k) {
                if (codes.size() >= 255) return fail(LBM_EINVAL, "more than 255 distinct forest codes");
                codes.push_back(c);
                k = (int)codes.size();
                tab[k] = (float)(h->Cd * forest_code_lad(c, a_fm));
            }
            last = c; last_k = k;
        }
        idx[n] = (uint8_t)k;
        frow[(n / h->nx) % h->ny] = 1;
    }
    CU_TRY(cudaMemcpyAsync(h->ws + h->L.fidx, idx.data(), (size_t)h->N, cudaMemcpyHostToDevice, h->stream));
    CU_TRY(cudaMemcpyAsync(h->ws + h->L.ftab, tab.data(), 256 * 4, cudaMemcpyHostToDevice, h->stream));
    CU_TRY(cudaMemcpyAsync(h->ws + h->L.frow, frow.data(), (size_t)h->ny, cudaMemcpyHostToDevice, h->stream));
    h->forest_codes = true;
    h->kp.fidx = reinterpret_cast<const unsigned char *>(h->ws + h->L.fidx);
    int rc = rebuild_block_flags(h);
    if (rc) return rc;
    CU_TRY(cudaStreamSynchronize(h->stream));
    return LBM_OK;
}

int lbm_set_top_velocity(lbm_t *h, const double *U_top)
{
    if (!h) return fail(LBM_EINVAL, "handle is NULL");
    DevGuard dg(h);
    if (!U_top) return fail(LBM_EINVAL, "U_top is NULL");
    if (h->top != BC_TOP_LID) return fail(LBM_EINVAL, "handle was not created with LBM_TOP_FORCED_EQ");
    for (int a = 0; a < 3; ++a)
        if (!std::isfinite(U_top[a])) return fail(LBM_EINVAL, "U_top[%d] is not finite", a);
    for (int a = 0; a < 3; ++a) h->Utop[a] = U_top[a];
    graph_drop(h);
    if (h->bound) fill_params(h);
    return LBM_OK;
}

int lbm_set_init(lbm_t *h, int kind, double U_ref, double noise_frac)
{
    if (!h) return fail(LBM_EINVAL, "handle is NULL");
    if (kind < 0 || kind > 2) return fail(LBM_EINVAL, "unknown init kind %d", kind);
    if (!std::isfinite(U_ref) || !std::isfinite(noise_frac)) return fail(LBM_EINVAL, "U_ref / noise_frac not finite");
    h->init_kind = kind; h->U_ref = U_ref; h->noise_frac = noise_frac;
    return LBM_OK;
}

// ---- launch helpers --------------------------------------------------------------------------

template <int V>
static cudaError_t launch_init_v(lbm_s *h, const KParams &p, int planes)
{
    dim3 block(h->TX, h->TY), grid((unsigned)((long long)planes * h->ny / h->TY * h->nchunk));
    if (h->mask) {
        if (h->aax) init_kernel<V, WR_XO, true><<<grid, block, 0, h->stream>>>(p);
        else if (h->aa) init_kernel<V, WR_PUSH, true><<<grid, block, 0, h->stream>>>(p);
        else init_kernel<V, WR_LOCAL, true><<<grid, block, 0, h->stream>>>(p);
    } else if (h->aax) init_kernel<V, WR_XO><<<grid, block, 0, h->stream>>>(p);
    else if (h->aa) init_kernel<V, WR_PUSH><<<grid, block, 0, h->stream>>>(p);
    else init_kernel<V, WR_LOCAL><<<grid, block, 0, h->stream>>>(p);
    h->launches++;
    return cudaGetLastError();
}
static cudaError_t launch_init(lbm_s *h, const KParams &p, int planes)
{
    switch (h->V) {
    case 4: return launch_init_v<4>(h, p, planes);
    case 2: return launch_init_v<2>(h, p, planes);
    default: return launch_init_v<1>(h, p, planes);
    }
}

template <int V>
static cudaError_t launch_macros_v(lbm_s *h, const KParams &p, int planes)
{
    dim3 block(h->TX, h->TY), grid((unsigned)((long long)planes * h->ny / h->TY * h->nchunk));
    if (h->mask) {
        if (!h->aa) macros_kernel<V, RD_PULL, true><<<grid, block, 0, h->stream>>>(p);
        else if (h->aax && (h->t & 1) == 0) macros_kernel<V, RD_XE, true><<<grid, block, 0, h->stream>>>(p);
        else if (h->aax) macros_kernel<V, RD_XO, true><<<grid, block, 0, h->stream>>>(p);
        else if ((h->t & 1) == 0) macros_kernel<V, RD_LOCAL, true><<<grid, block, 0, h->stream>>>(p);
        else macros_kernel<V, RD_PULL_OPP, true><<<grid, block, 0, h->stream>>>(p);
    } else if (!h->aa) macros_kernel<V, RD_PULL><<<grid, block, 0, h->stream>>>(p);
    else if (h->aax && (h->t & 1) == 0) macros_kernel<V, RD_XE><<<grid, block, 0, h->stream>>>(p);
    else if (h->aax) macros_kernel<V, RD_XO><<<grid, block, 0, h->stream>>>(p);
    else if ((h->t & 1) == 0) macros_kernel<V, RD_LOCAL><<<grid, block, 0, h->stream>>>(p);
    else macros_kernel<V, RD_PULL_OPP><<<grid, block, 0, h->stream>>>(p);
    h->launches++;
    return cudaGetLastError();
}
static cudaError_t launch_macros(lbm_s *h, const KParams &p, int planes)
{
    switch (h->V) {
    case 4: return launch_macros_v<4>(h, p, planes);
    case 2: return launch_macros_v<2>(h, p, planes);
    default: return launch_macros_v<1>(h, p, planes);
    }
}

static bool pdl_enabled()
{
    static const int on = [] { const char *e = getenv("LBM_PDL"); return (e && *e) ? atoi(e) : 1; }();   // A-B switch
    return on != 0;
}

// One launch of the fused step for the planes [p.z0, p.z1): the launchers live in their own
// translation units (lbm_launch.cuh), one per (cells per thread, statistics, SGS row table).
static cudaError_t launch_step(lbm_s *h, const KParams &p, bool stats)
{
    StepLaunch L;
    L.TX = h->TX; L.TY = h->TY; L.nchunk = h->nchunk; L.nx = h->nx; L.ny = h->ny;
    L.mask = h->mask && h->nflagged > 0;      // nothing flagged: the plain kernels
    L.aa = h->aa; L.aax = h->aax; L.odd = (h->t & 1) != 0;
    L.tma_mode = h->tma_mode; L.tma_rows = h->tma_rows;
    {
        static const int g3 = [] { const char *e = getenv("LBM_GRID3"); return (e && *e) ? atoi(e) : 1; }();   // A-B switch
        L.grid3 = g3 != 0;
        L.pdl = pdl_enabled();
    }
    // the map of the array this step reads (two-lattice: the roles swap every step)
    const bool swapped = !h->aa && p.src != reinterpret_cast<float *>(h->ws + h->L.pops);
    L.map = swapped ? &h->map_b : &h->map_a;
    L.stream = h->stream;
    const bool sgs = p.sgs != nullptr;
    h->launches++;
    if (h->V == 4 && h->tma_mode && !sgs) {
        const cudaError_t e = stats ? launch_tma_t<true>(L, p) : launch_tma_t<false>(L, p);
        if (e != cudaErrorNotSupported) return e;
    }
#define LBM_GO(V) \
    return stats ? (sgs ? launch_step_t<V, true, true>(L, p) : launch_step_t<V, true, false>(L, p)) \
                 : (sgs ? launch_step_t<V, false, true>(L, p) : launch_step_t<V, false, false>(L, p));
    switch (h->V) {
    case 4: LBM_GO(4)
    case 2: LBM_GO(2)
    default: LBM_GO(1)
    }
#undef LBM_GO
}

static cudaError_t launch_stage2(lbm_s *h, int mode)
{
    dim3 grid(h->ny, NSTAT);
    h->launches++;
    return launch_chain(stats_stage2_kernel, grid, dim3(256), 0, h->stream, pdl_enabled(),
        reinterpret_cast<const float *>(h->ws + h->L.partial), (long long)h->nz * h->pchunks,
        reinterpret_cast<double *>(h->ws + h->L.acc), reinterpret_cast<float *>(h->ws + h->L.shift), mode,
        1.0 / ((double)h->nx * h->nz), reinterpret_cast<int *>(h->ws + h->L.flag));
}

static int stats_reset_impl(lbm_s *h)
{
    CU_TRY(cudaMemsetAsync(h->ws + h->L.acc, 0, (size_t)h->ny * NSTAT * 8, h->stream));
    CU_TRY(cudaMemsetAsync(h->ws + h->L.shift, 0, (size_t)h->ny * 16, h->stream));
    CU_TRY(cudaMemsetAsync(h->ws + h->L.flag, 0, 256, h->stream));
    h->nsamples = 0; h->stats_phase = 0;
    if (h->inited && !h->mask && !h->halo) {
        // centre the accumulation on the current plane means (numerical shift only; not with a
        // solid mask, where the number of contributing cells differs from thread to thread)
        KParams p = h->kp;
        p.partial = reinterpret_cast<float *>(h->ws + h->L.partial);
        p.shift = nullptr;
        CU_TRY(launch_macros(h, p, h->nz));
        CU_TRY(launch_stage2(h, 1));
    }
    return LBM_OK;
}

// r_j = J0_j / 12 with 16 significant bits, so that 2 r (axis populations) and 12 r (= J0) are
// exact in fp32 (kernels: mom_ref_shift).
static int upload_reference(lbm_s *h, const double *jx_ref)
{
    std::vector<float> r(h->ny, 0.f);
    if (jx_ref)
        for (int j = 0; j < h->ny; ++j) {
            float v = (float)(jx_ref[j] / 12.0);
            uint32_t b;
            memcpy(&b, &v, 4);
            b &= 0xFFFFFF00u;
            memcpy(&v, &b, 4);
            r[j] = std::isfinite(v) ? v : 0.f;
        }
    graph_drop(h);
    CU_TRY(cudaMemcpyAsync(h->ws + h->L.jref, r.data(), h->ny * 4, cudaMemcpyHostToDevice, h->stream));
    CU_TRY(cudaStreamSynchronize(h->stream));
    return LBM_OK;
}

int lbm_set_reference_profile(lbm_t *h, const double *jx_ref_host)
{
    if (!h) return fail(LBM_EINVAL, "handle is NULL");
    DevGuard dg(h);
    if (!h->bound) return fail(LBM_ESTATE, "lbm_set_reference_profile before lbm_bind");
    if (jx_ref_host)
        for (int j = 0; j < h->ny; ++j)
            if (!std::isfinite(jx_ref_host[j])) return fail(LBM_EINVAL, "jx_ref[%d] is not finite", j);
    return upload_reference(h, jx_ref_host);
}

int lbm_get_reference_profile(lbm_t *h, double *jx_ref_host)
{
    if (!h) return fail(LBM_EINVAL, "handle is NULL");
    DevGuard dg(h);
    if (!h->bound) return fail(LBM_ESTATE, "lbm_get_reference_profile before lbm_bind");
    if (!jx_ref_host) return fail(LBM_EINVAL, "output is NULL");
    std::vector<float> r(h->ny);
    CU_TRY(cudaMemcpyAsync(r.data(), h->ws + h->L.jref, h->ny * 4, cudaMemcpyDeviceToHost, h->stream));
    CU_TRY(cudaStreamSynchronize(h->stream));
    for (int j = 0; j < h->ny; ++j) jx_ref_host[j] = 12.0 * (double)r[j];
    return LBM_OK;
}

static int upload_profile(lbm_s *h)
{
    std::vector<float> up(h->ny);
    for (int j = 0; j < h->ny; ++j) {
        const double eta = (j + 0.5) / h->ny;
        double U = 0.0;
        if (h->init_kind == LBM_INIT_POWER_LAW) U = h->U_ref * std::pow(eta, 1.0 / 7.0);
        else if (h->init_kind == LBM_INIT_PARABOLA) U = h->U_ref * 4.0 * eta * (1.0 - eta);
        up[j] = (float)U;
    }
    CU_TRY(cudaMemcpyAsync(h->ws + h->L.uprof, up.data(), h->ny * 4, cudaMemcpyHostToDevice, h->stream));
    CU_TRY(cudaStreamSynchronize(h->stream));
    // the synthetic profile (rho = 1) is also the momentum reference of the run it starts
    std::vector<double> ref(up.begin(), up.end());
    return upload_reference(h, ref.data());
}

int lbm_init(lbm_t *h, uint64_t seed)
{
    if (!h) return fail(LBM_EINVAL, "handle is NULL");
    DevGuard dg(h);
    if (!h->bound) return fail(LBM_ESTATE, "lbm_init before lbm_bind");
    int rc = upload_profile(h);
    if (rc) return rc;
    fill_params(h);
    KParams p = h->kp;
    p.rho_in = nullptr; p.u_in = nullptr;
    p.noise_amp = h->noise_frac * h->U_ref;
    p.seed = seed;
    p.dst = p.src; // state 0 lives in the primary array
    CU_TRY(launch_init(h, p, h->nz));
    h->t = 0; h->inited = true;
    return stats_reset_impl(h);
}

int lbm_set_macros(lbm_t *h, const float *rho_dev, const float *u_dev)
{
    if (!h) return fail(LBM_EINVAL, "handle is NULL");
    DevGuard dg(h);
    if (!h->bound) return fail(LBM_ESTATE, "lbm_set_macros before lbm_bind");
    if (!rho_dev || !u_dev) return fail(LBM_EINVAL, "rho / u is NULL");
    fill_params(h);
    KParams p = h->kp;
    p.rho_in = rho_dev; p.u_in = u_dev; p.dst = p.src;
    CU_TRY(launch_init(h, p, h->nz));
    h->t = 0; h->inited = true;
    return stats_reset_impl(h);
}

int lbm_set_macros_host(lbm_t *h, const float *rho_host, const float *u_host)
{
    if (!h) return fail(LBM_EINVAL, "handle is NULL");
    DevGuard dg(h);
    if (!h->bound) return fail(LBM_ESTATE, "lbm_set_macros_host before lbm_bind");
    if (!rho_host || !u_host) return fail(LBM_EINVAL, "rho / u is NULL");
    fill_params(h);
    const size_t plane = (size_t)h->nx * h->ny;
    float *stg = reinterpret_cast<float *>(h->ws + h->L.staging);
    for (int z0 = 0; z0 < h->nz; z0 += h->L.stage_planes) {
        const int zc = (h->nz - z0 < h->L.stage_planes) ? h->nz - z0 : h->L.stage_planes;
        const size_t cnt = plane * zc;
        CU_TRY(cudaMemcpyAsync(stg, rho_host + plane * z0, cnt * 4, cudaMemcpyHostToDevice, h->stream));
        for (int a = 0; a < 3; ++a)
            CU_TRY(cudaMemcpyAsync(stg + cnt * (1 + a), u_host + (size_t)h->N * a + plane * z0, cnt * 4,
                                   cudaMemcpyHostToDevice, h->stream));
        KParams p = h->kp;
        p.rho_in = stg; p.u_in = stg + cnt; p.Nio = (long long)cnt; p.zoff = 0;
        p.z0 = z0; p.z1 = z0 + zc; p.dst = p.src;
        CU_TRY(launch_init(h, p, zc));
    }
    h->t = 0; h->inited = true;
    int rc = stats_reset_impl(h);
    if (rc) return rc;
    CU_TRY(cudaStreamSynchronize(h->stream));
    return LBM_OK;
}

// one step-kernel launch, bracketed by a pair of events when kernel timing is on
static int launch_step_timed(lbm_s *h, const KParams &p, bool sample)
{
    const bool timed = h->timing && h->ev_used + 2 <= 2 * MAX_TIMED;
    if (timed) {
        while (h->ev.size() < h->ev_used + 2) {
            cudaEvent_t e;
            CU_TRY(cudaEventCreate(&e));
            h->ev.push_back(e);
        }
        CU_TRY(cudaEventRecord(h->ev[h->ev_used], h->stream));
    }
    CU_TRY(launch_step(h, p, sample));
    if (timed) {
        CU_TRY(cudaEventRecord(h->ev[h->ev_used + 1], h->stream));
        h->ev_used += 2;
    }
    return LBM_OK;
}

// parameters of the step that maps state t -> t+1
static KParams step_params(lbm_s *h, bool sample)
{
    KParams p = h->kp;
    if (!h->aa && (h->t & 1)) { float *t = p.src; p.src = p.dst; p.dst = t; }
    p.z0 = h->zlo; p.z1 = h->zhi;
    p.rev = h->sweep ? (int)(h->t & 1) : 0;
    if (sample) {
        p.partial = reinterpret_cast<float *>(h->ws + h->L.partial);
        p.shift = (h->mask || h->halo) ? nullptr : reinterpret_cast<const float *>(h->ws + h->L.shift);
    }
    return p;
}

// n time steps, one launch (+ the stage-2 launch on sampled steps) each
static int step_direct(lbm_s *h, int n)
{
    for (int k = 0; k < n; ++k) {
        const bool sample = h->stats_every > 0 && (h->stats_phase % h->stats_every) == 0;
        const KParams p = step_params(h, sample);
        int rc = launch_step_timed(h, p, sample);
        if (rc) return rc;
        if (sample) {
            CU_TRY(launch_stage2(h, 0));
            h->nsamples++;
        }
        if (h->stats_every > 0) h->stats_phase++;
        h->t++;
    }
    return LBM_OK;
}

// Steps per graph: a whole number of periods of (storage parity x sampling cadence), about 32
// steps; 0 = this cadence is not worth a graph.
static int graph_span(const lbm_s *h)
{
    const int e = h->stats_every;
    const int period = (e == 0) ? 2 : ((e % 2 == 0) ? e : 2 * e);
    if (period > 64) return 0;
    int reps = 32 / period;
    if (reps < 1) reps = 1;
    return period * reps;
}

// Capture G steps starting at the current parity (sampling phase 0) into an executable graph.
// Returns LBM_OK with h->gexec == nullptr when the stream cannot be captured (e.g. the caller
// is capturing it already): the caller then falls back to direct launches.
static int graph_build(lbm_s *h, int G)
{
    graph_drop(h);
    cudaStreamCaptureStatus cs = cudaStreamCaptureStatusNone;
    if (cudaStreamIsCapturing(h->stream, &cs) != cudaSuccess || cs != cudaStreamCaptureStatusNone) {
        cudaGetLastError();
        return LBM_OK;
    }
    const long long t0 = h->t, ph0 = h->stats_phase, ns0 = h->nsamples, l0 = h->launches;
    if (cudaStreamBeginCapture(h->stream, cudaStreamCaptureModeThreadLocal) != cudaSuccess) {
        cudaGetLastError();
        return LBM_OK;
    }
    const int rc = step_direct(h, G);
    cudaGraph_t graph = nullptr;
    const cudaError_t e = cudaStreamEndCapture(h->stream, &graph);
    h->g_launches = h->launches - l0; h->g_samples = h->nsamples - ns0;
    h->t = t0; h->stats_phase = ph0; h->nsamples = ns0; h->launches = l0;   // nothing has run yet
    if (rc != LBM_OK || e != cudaSuccess || !graph) {
        cudaGetLastError();
        if (graph) cudaGraphDestroy(graph);
        return LBM_OK;
    }
    if (cudaGraphInstantiate(&h->gexec, graph, 0) != cudaSuccess) { cudaGetLastError(); h->gexec = nullptr; }
    cudaGraphDestroy(graph);
    h->g_steps = G; h->g_parity = (int)(t0 & 1); h->g_every = h->stats_every;
    return LBM_OK;
}

int lbm_step(lbm_t *h, int n)
{
    if (!h) return fail(LBM_EINVAL, "handle is NULL");
    DevGuard dg(h);
    if (!h->inited) return fail(LBM_ESTATE, "lbm_step before lbm_init / lbm_set_macros");
    if (n < 0) return fail(LBM_EINVAL, "n must be >= 0");
    // small lattices are launch-bound: replay G steps as one CUDA graph (identical kernels and
    // order, so results are bit-identical to direct launches)
    const bool want = h->graph_mode == 1 || (h->graph_mode == 2 && h->N <= (1ll << 22));
    const int G = (want && !h->timing) ? graph_span(h) : 0;
    if (G > 0 && n >= 2 * G) {
        if (h->stats_every > 0) {            // align the sampling phase first
            const int mis = (int)(h->stats_phase % h->stats_every);
            if (mis) { const int a = h->stats_every - mis; int rc = step_direct(h, a); if (rc) return rc; n -= a; }
        }
        if (n >= G) {
            if (!h->gexec || h->g_steps != G || h->g_parity != (int)(h->t & 1) || h->g_every != h->stats_every) {
                int rc = graph_build(h, G);
                if (rc) return rc;
            }
            while (h->gexec && n >= G) {
                CU_TRY(cudaGraphLaunch(h->gexec, h->stream));
                h->t += G; h->launches += h->g_launches; h->nsamples += h->g_samples;
                if (h->stats_every > 0) h->stats_phase += G;
                n -= G;
            }
        }
    }
    return step_direct(h, n);
}

int lbm_set_z_slab(lbm_t *h, int z_first, int nz_global)
{
    if (!h) return fail(LBM_EINVAL, "handle is NULL");
    if (!h->halo) return fail(LBM_EINVAL, "handle was not created with LBM_Z_HALO");
    if (nz_global < 1 || z_first < 0 || z_first >= nz_global) return fail(LBM_EINVAL, "bad slab position");
    h->zg0 = z_first - 1; h->nzg = nz_global;
    h->kp.zg0 = h->zg0; h->kp.nzg = h->nzg;
    return LBM_OK;
}

int lbm_halo_bytes(const lbm_t *h, size_t *bytes)
{
    if (!h || !bytes) return fail(LBM_EINVAL, "NULL argument");
    *bytes = (size_t)5 * h->nx * h->ny * 4;
    return LBM_OK;
}

// Which plane and which slot set (1: c_z = +1, 0: c_z = -1) a face of a slab in state t moves.
//   two-lattice        : populations leave from the boundary planes and enter the ghost planes;
//   single array, t odd : every population sits in the opposite slot of its own cell - the same
//                        planes, the opposite slot sets;
//   single array, t even: population i of cell x sits at slot i of cell x + c_i - what leaves has
//                        been pushed into the ghost planes and enters the neighbour's boundary plane
//                        (filtered: halo_kernel).
struct HaloMap { int z, slots; bool filter; };
static HaloMap halo_map(const lbm_s *h, long long t, int face, bool pack)
{
    const int nz = h->nz;
    if (!h->aa) return pack ? HaloMap{face ? nz - 2 : 1, face, false} : HaloMap{face ? nz - 1 : 0, face ? 0 : 1, false};
    if (t & 1) return pack ? HaloMap{face ? nz - 2 : 1, face ? 0 : 1, false} : HaloMap{face ? nz - 1 : 0, face, false};
    return pack ? HaloMap{face ? nz - 1 : 0, face, false} : HaloMap{face ? nz - 2 : 1, face ? 0 : 1, true};
}

// pack / unpack one face (face = 0, 1) or both (face = 2; buf = low-face buffer, buf_hi = high-face
// buffer) of the array `arr` holding state t: one launch, chained like the step kernels
static cudaError_t halo_launch(lbm_s *h, float *arr, long long t, int face, float *buf, bool pack, float *buf_hi = nullptr)
{
    const bool both = face == 2;
    const HaloMap m0 = halo_map(h, t, both ? 0 : face, pack), m1 = halo_map(h, t, 1, pack);
    const long long plane = (long long)h->nx * h->ny;
    const dim3 grid((unsigned)((5 * plane + 255) / 256), both ? 2u : 1u), block(256);
    const HaloFace f0{m0.z, m0.slots, buf}, f1{m1.z, m1.slots, buf_hi};
    h->launches++;
    const bool pdl = pdl_enabled();
    if (pack) return launch_chain(halo_kernel<true, false>, grid, block, 0, h->stream, pdl, h->kp, arr, f0, f1);
    if (m0.filter) return launch_chain(halo_kernel<false, true>, grid, block, 0, h->stream, pdl, h->kp, arr, f0, f1);
    return launch_chain(halo_kernel<false, false>, grid, block, 0, h->stream, pdl, h->kp, arr, f0, f1);
}

static int halo_copy(lbm_s *h, int side, float *buf, bool pack)
{
    if (!h) return fail(LBM_EINVAL, "handle is NULL");
    DevGuard dg(h);
    if (!h->halo) return fail(LBM_EINVAL, "handle was not created with LBM_Z_HALO");
    if (!h->inited) return fail(LBM_ESTATE, "halo call before lbm_init / lbm_set_macros");
    if (!buf || (side != 0 && side != 1)) return fail(LBM_EINVAL, "bad halo arguments");
    KParams p = h->kp;
    if (!h->aa && (h->t & 1)) { float *t = p.src; p.src = p.dst; p.dst = t; }   // the lattice holding state t
    CU_TRY(halo_launch(h, p.src, h->t, side, buf, pack));
    return LBM_OK;
}

int lbm_halo_pack(lbm_t *h, int side, float *buf_dev) { return halo_copy(h, side, buf_dev, true); }
int lbm_halo_unpack(lbm_t *h, int side, const float *buf_dev)
{
    return halo_copy(h, side, const_cast<float *>(buf_dev), false);
}

// One time step of a z slab, split so that the halo exchange overlaps the interior update:
//   begin: update the two boundary planes, pack the faces of the NEW state, record `packed`,
//          then launch the update of the interior planes;
//   (caller: on another stream, wait for `packed`, exchange the buffers with the ring
//    neighbours, record `ready`)
//   end:   wait for `ready`, unpack into the ghost planes of the new state, statistics stage 2.
int lbm_step_slab_begin(lbm_t *h, float *send_lo_dev, float *send_hi_dev, void *packed_event)
{
    if (!h) return fail(LBM_EINVAL, "handle is NULL");
    DevGuard dg(h);
    if (!h->halo) return fail(LBM_EINVAL, "handle was not created with LBM_Z_HALO");
    if (!h->inited) return fail(LBM_ESTATE, "lbm_step_slab_begin before lbm_init / lbm_set_macros");
    if (h->slab_open) return fail(LBM_ESTATE, "lbm_step_slab_begin twice without lbm_step_slab_end");
    if (!send_lo_dev || !send_hi_dev) return fail(LBM_EINVAL, "send buffer is NULL");
    const bool sample = h->stats_every > 0 && (h->stats_phase % h->stats_every) == 0;
    KParams p = step_params(h, sample);
    const int zl = h->zlo, zh = h->zhi;                   // interior planes [1, nz-1)
    int rc;
    p.z0 = zl; p.z1 = zl + 1;
    if ((rc = launch_step_timed(h, p, sample))) return rc;
    if (zh - 1 > zl) {
        p.z0 = zh - 1; p.z1 = zh;
        if ((rc = launch_step_timed(h, p, sample))) return rc;
    }
    CU_TRY(halo_launch(h, p.dst, h->t + 1, 2, send_lo_dev, true, send_hi_dev));      // p.dst holds state t+1
    if (packed_event) CU_TRY(cudaEventRecord(static_cast<cudaEvent_t>(packed_event), h->stream));
    if (zh - 1 > zl + 1) {
        p.z0 = zl + 1; p.z1 = zh - 1;
        if ((rc = launch_step_timed(h, p, sample))) return rc;
    }
    h->slab_open = true; h->slab_sample = sample;
    return LBM_OK;
}

int lbm_step_slab_end(lbm_t *h, const float *recv_lo_dev, const float *recv_hi_dev, void *ready_event)
{
    if (!h) return fail(LBM_EINVAL, "handle is NULL");
    DevGuard dg(h);
    if (!h->halo) return fail(LBM_EINVAL, "handle was not created with LBM_Z_HALO");
    if (!h->slab_open) return fail(LBM_ESTATE, "lbm_step_slab_end without lbm_step_slab_begin");
    if (!recv_lo_dev || !recv_hi_dev) return fail(LBM_EINVAL, "receive buffer is NULL");
    if (ready_event) CU_TRY(cudaStreamWaitEvent(h->stream, static_cast<cudaEvent_t>(ready_event), 0));
    const KParams p = step_params(h, false);              // p.dst holds state t+1
    // what entered through the low face comes from the lower neighbour's high face and vice versa
    CU_TRY(halo_launch(h, p.dst, h->t + 1, 2, const_cast<float *>(recv_lo_dev), false, const_cast<float *>(recv_hi_dev)));
    if (h->slab_sample) {
        CU_TRY(launch_stage2(h, 0));
        h->nsamples++;
    }
    if (h->stats_every > 0) h->stats_phase++;
    h->t++;
    h->slab_open = false;
    return LBM_OK;
}

int lbm_stats_read_raw(lbm_t *h, double *out, double *centre, double *count)
{
    if (!h) return fail(LBM_EINVAL, "handle is NULL");
    DevGuard dg(h);
    if (!h->bound) return fail(LBM_ESTATE, "lbm_stats_read_raw before lbm_bind");
    if (!out) return fail(LBM_EINVAL, "out is NULL");
    std::vector<float> shift((size_t)h->ny * 4);
    int flag = 0;
    CU_TRY(cudaMemcpyAsync(out, h->ws + h->L.acc, (size_t)h->ny * NSTAT * 8, cudaMemcpyDeviceToHost, h->stream));
    CU_TRY(cudaMemcpyAsync(shift.data(), h->ws + h->L.shift, shift.size() * 4, cudaMemcpyDeviceToHost, h->stream));
    CU_TRY(cudaMemcpyAsync(&flag, h->ws + h->L.flag, 4, cudaMemcpyDeviceToHost, h->stream));
    CU_TRY(cudaStreamSynchronize(h->stream));
    for (int y = 0; y < h->ny; ++y) {
        out[(size_t)y * NSTAT + 9] += (double)h->nsamples * h->nfluid[y];   // sum of rho, not of rho-1
        if (centre) for (int a = 0; a < 3; ++a) centre[y * 3 + a] = shift[y * 4 + a];
    }
    if (count) *count = (double)h->nsamples * h->nx * (h->zhi - h->zlo);
    if (flag) return fail(LBM_EDIVERGED, "non-finite plane sum of rho seen by the statistics reduction");
    return LBM_OK;
}

int lbm_stats_from_raw(const double *raw, const double *centre, int ny, double count, double *out)
{
    if (!raw || !out || ny < 1) return fail(LBM_EINVAL, "bad arguments");
    for (int y = 0; y < ny; ++y) {
        const double *a = raw + (size_t)y * NSTAT;
        double *r = out + (size_t)y * NSTAT;
        if (!(count > 0.0)) { for (int k = 0; k < NSTAT; ++k) r[k] = 0.0; continue; }
        const double mu = a[0] / count, mv = a[1] / count, mw = a[2] / count;
        r[0] = mu + (centre ? centre[y * 3 + 0] : 0.0);
        r[1] = mv + (centre ? centre[y * 3 + 1] : 0.0);
        r[2] = mw + (centre ? centre[y * 3 + 2] : 0.0);
        r[3] = a[3] / count - mu * mu; r[4] = a[4] / count - mv * mv; r[5] = a[5] / count - mw * mw;
        r[6] = a[6] / count - mu * mv; r[7] = a[7] / count - mv * mw; r[8] = a[8] / count - mu * mw;
        r[9] = a[9] / count;
    }
    return LBM_OK;
}

int lbm_set_tma(lbm_t *h, int mode, int rows)
{
    if (!h) return fail(LBM_EINVAL, "handle is NULL");
    DevGuard dg(h);
    if (mode < 0 || mode > 7) return fail(LBM_EINVAL, "mode is a bit mask 0..7");
    if (mode && !h->tma_ok)
        return fail(LBM_EINVAL, "the TMA path needs 4 cells per thread, nx %% 256 == 0 and no solid mask");
    if (rows != 0 && !((rows == 1 || rows == 2 || rows == 4) && h->ny % rows == 0))
        return fail(LBM_EINVAL, "rows per tile must be 1, 2 or 4 and divide ny");
    graph_drop(h);
    h->tma_mode = mode;
    if (rows) h->tma_rows = rows;
    set_variant(h);
    return set_pchunks(h);
}

// Row-table SGS models: tau_total = max(tau0, (t + sqrt(t^2 + 18 sqrt(2) C_j Q^{1/2} / rho)) / 2) with
// t = tau0 - 3 C_j Sbar_j; the table holds {t, 18 sqrt(2) C_j} per row.
int lbm_set_sgs_rows(lbm_t *h, const double *csmag_row_host, const double *sbar_row_host)
{
    if (!h) return fail(LBM_EINVAL, "handle is NULL");
    DevGuard dg(h);
    if (!h->bound) return fail(LBM_ESTATE, "lbm_set_sgs_rows before lbm_bind");
    graph_drop(h);
    if (!csmag_row_host && !sbar_row_host) {
        h->sgs_rows = false; h->kp.sgs = nullptr;
        return LBM_OK;
    }
    const double tau0 = 3.0 * h->nu + 0.5;
    std::vector<float> tab((size_t)h->ny * 2);
    for (int j = 0; j < h->ny; ++j) {
        const double C = csmag_row_host ? csmag_row_host[j] : h->Cs * h->Cs;
        const double S = sbar_row_host ? sbar_row_host[j] : 0.0;
        if (!(C >= 0.0) || !std::isfinite(C)) return fail(LBM_EINVAL, "csmag_row[%d] must be >= 0", j);
        if (!(S >= 0.0) || !std::isfinite(S)) return fail(LBM_EINVAL, "sbar_row[%d] must be >= 0", j);
        tab[2 * j] = (float)(tau0 - 3.0 * C * S);
        tab[2 * j + 1] = (float)(18.0 * std::sqrt(2.0) * C);
    }
    CU_TRY(cudaMemcpyAsync(h->ws + h->L.sgs, tab.data(), tab.size() * 4, cudaMemcpyHostToDevice, h->stream));
    CU_TRY(cudaStreamSynchronize(h->stream));     // tab is a local vector
    h->sgs_rows = true;
    h->kp.sgs = reinterpret_cast<const float2 *>(h->ws + h->L.sgs);
    return LBM_OK;
}

int lbm_sgs_van_driest(int ny, double Cs, double u_tau, double nu, double A_plus, int both_walls, double *csmag_row_out)
{
    if (ny < 1 || !csmag_row_out) return fail(LBM_EINVAL, "bad arguments");
    if (!(Cs >= 0.0) || !(u_tau >= 0.0) || !(nu > 0.0) || !(A_plus > 0.0)) return fail(LBM_EINVAL, "Cs, u_tau >= 0 and nu, A_plus > 0 are required");
    for (int j = 0; j < ny; ++j) {
        double dist = j + 0.5;                                  // cell centre to the bottom wall face
        if (both_walls) dist = std::fmin(dist, (double)ny - dist);
        const double damp = -std::expm1(-dist * u_tau / (nu * A_plus));   // 1 - exp(-y+/A+)
        csmag_row_out[j] = Cs * Cs * damp * damp;
    }
    return LBM_OK;
}

int lbm_sgs_mean_shear(const double *stats, int ny, int top_wall, double *sbar_row_out)
{
    if (!stats || ny < 1 || !sbar_row_out) return fail(LBM_EINVAL, "bad arguments");
    auto prof = [&](int j, int col) {       // profile extended past the faces: odd image at a wall, even otherwise
        if (j < 0) return -stats[col];
        if (j >= ny) return (top_wall ? -1.0 : 1.0) * stats[(size_t)(ny - 1) * NSTAT + col];
        return stats[(size_t)j * NSTAT + col];
    };
    for (int j = 0; j < ny; ++j) {
        const double du = 0.5 * (prof(j + 1, 0) - prof(j - 1, 0)), dw = 0.5 * (prof(j + 1, 2) - prof(j - 1, 2));
        sbar_row_out[j] = std::hypot(du, dw);
    }
    return LBM_OK;
}

int lbm_set_sweep(lbm_t *h, int mode)
{
    if (!h) return fail(LBM_EINVAL, "handle is NULL");
    if (mode != 0 && mode != 1) return fail(LBM_EINVAL, "mode must be 0 (forward) or 1 (alternating)");
    DevGuard dg(h);
    graph_drop(h);
    h->sweep = mode;
    return LBM_OK;
}

int lbm_set_graphs(lbm_t *h, int mode)
{
    if (!h) return fail(LBM_EINVAL, "handle is NULL");
    DevGuard dg(h);
    if (mode < 0 || mode > 2) return fail(LBM_EINVAL, "mode must be 0 (off), 1 (on) or 2 (auto)");
    h->graph_mode = mode;
    if (mode == 0) graph_drop(h);
    return LBM_OK;
}

// current read-side parameters (two-lattice: the array holding state t)
static KParams read_params(lbm_s *h)
{
    KParams p = h->kp;
    if (!h->aa && (h->t & 1)) { float *t = p.src; p.src = p.dst; p.dst = t; }
    return p;
}

int lbm_get_macros(lbm_t *h, float *rho_dev, float *u_dev)
{
    if (!h) return fail(LBM_EINVAL, "handle is NULL");
    DevGuard dg(h);
    if (!h->inited) return fail(LBM_ESTATE, "lbm_get_macros before lbm_init / lbm_set_macros");
    KParams p = read_params(h);
    p.rho_out = rho_dev; p.u_out = u_dev;
    CU_TRY(launch_macros(h, p, h->nz));
    return LBM_OK;
}

int lbm_get_macros_host(lbm_t *h, float *rho_host, float *u_host)
{
    if (!h) return fail(LBM_EINVAL, "handle is NULL");
    DevGuard dg(h);
    if (!h->inited) return fail(LBM_ESTATE, "lbm_get_macros_host before lbm_init / lbm_set_macros");
    const size_t plane = (size_t)h->nx * h->ny;
    float *stg = reinterpret_cast<float *>(h->ws + h->L.staging);
    for (int z0 = 0; z0 < h->nz; z0 += h->L.stage_planes) {
        const int zc = (h->nz - z0 < h->L.stage_planes) ? h->nz - z0 : h->L.stage_planes;
        const size_t cnt = plane * zc;
        KParams p = read_params(h);
        p.rho_out = rho_host ? stg : nullptr;
        p.u_out = u_host ? stg + cnt : nullptr;
        p.Nio = (long long)cnt; p.zoff = 0; p.z0 = z0; p.z1 = z0 + zc;
        CU_TRY(launch_macros(h, p, zc));
        if (rho_host)
            CU_TRY(cudaMemcpyAsync(rho_host + plane * z0, stg, cnt * 4, cudaMemcpyDeviceToHost, h->stream));
        if (u_host)
            for (int a = 0; a < 3; ++a)
                CU_TRY(cudaMemcpyAsync(u_host + (size_t)h->N * a + plane * z0, stg + cnt * (1 + a), cnt * 4,
                                       cudaMemcpyDeviceToHost, h->stream));
    }
    int flag = 0;
    CU_TRY(cudaMemcpyAsync(&flag, h->ws + h->L.flag, 4, cudaMemcpyDeviceToHost, h->stream));
    CU_TRY(cudaStreamSynchronize(h->stream));
    if (flag) return fail(LBM_EDIVERGED, "non-finite density in the sampled field");
    return LBM_OK;
}

int lbm_diverged(lbm_t *h, int *flag_out)
{
    if (!h) return fail(LBM_EINVAL, "handle is NULL");
    DevGuard dg(h);
    if (!h->bound) return fail(LBM_ESTATE, "lbm_diverged before lbm_bind");
    int flag = 0;
    CU_TRY(cudaMemcpyAsync(&flag, h->ws + h->L.flag, 4, cudaMemcpyDeviceToHost, h->stream));
    CU_TRY(cudaStreamSynchronize(h->stream));
    if (flag_out) *flag_out = flag;
    if (flag) return fail(LBM_EDIVERGED, "a non-finite density was seen by lbm_get_macros* or the statistics reduction");
    return LBM_OK;
}

int lbm_get_state(lbm_t *h, float *out_dev)
{
    if (!h) return fail(LBM_EINVAL, "handle is NULL");
    DevGuard dg(h);
    if (!h->inited) return fail(LBM_ESTATE, "lbm_get_state before lbm_init / lbm_set_macros");
    if (!out_dev) return fail(LBM_EINVAL, "output is NULL");
    KParams p = read_params(h);
    const unsigned blocks = (unsigned)((h->N + 255) / 256);
    if (!h->aa) state_kernel<0><<<blocks, 256, 0, h->stream>>>(p, out_dev);
    else if (h->aax && (h->t & 1)) state_kernel<3><<<blocks, 256, 0, h->stream>>>(p, out_dev);
    else if (h->aax) state_kernel<4><<<blocks, 256, 0, h->stream>>>(p, out_dev);
    else if (h->t & 1) state_kernel<1><<<blocks, 256, 0, h->stream>>>(p, out_dev);
    else state_kernel<2><<<blocks, 256, 0, h->stream>>>(p, out_dev);
    h->launches++;
    CU_TRY(cudaGetLastError());
    return LBM_OK;
}

template <int V>
static cudaError_t launch_setstate_v(lbm_s *h, const KParams &p, const float *in, bool odd)
{
    dim3 block(h->TX, h->TY), grid((unsigned)((long long)h->nz * h->ny / h->TY * h->nchunk));
    if (h->mask) {
        if (!h->aa) setstate_kernel<V, WR_LOCAL, true><<<grid, block, 0, h->stream>>>(p, in);
        else if (h->aax && odd) setstate_kernel<V, WR_XE, true><<<grid, block, 0, h->stream>>>(p, in);
        else if (h->aax) setstate_kernel<V, WR_XO, true><<<grid, block, 0, h->stream>>>(p, in);
        else if (odd) setstate_kernel<V, WR_LOCAL_OPP, true><<<grid, block, 0, h->stream>>>(p, in);
        else setstate_kernel<V, WR_PUSH, true><<<grid, block, 0, h->stream>>>(p, in);
    } else if (!h->aa) setstate_kernel<V, WR_LOCAL><<<grid, block, 0, h->stream>>>(p, in);
    else if (h->aax && odd) setstate_kernel<V, WR_XE><<<grid, block, 0, h->stream>>>(p, in);
    else if (h->aax) setstate_kernel<V, WR_XO><<<grid, block, 0, h->stream>>>(p, in);
    else if (odd) setstate_kernel<V, WR_LOCAL_OPP><<<grid, block, 0, h->stream>>>(p, in);
    else setstate_kernel<V, WR_PUSH><<<grid, block, 0, h->stream>>>(p, in);
    h->launches++;
    return cudaGetLastError();
}

int lbm_set_state(lbm_t *h, const float *in_dev, long long t)
{
    if (!h) return fail(LBM_EINVAL, "handle is NULL");
    DevGuard dg(h);
    if (!h->bound) return fail(LBM_ESTATE, "lbm_set_state before lbm_bind");
    if (!in_dev) return fail(LBM_EINVAL, "input is NULL");
    if (t < 0) return fail(LBM_EINVAL, "t must be >= 0");
    fill_params(h);
    KParams p = h->kp;
    const bool odd = (t & 1) != 0;
    if (!h->aa && odd) p.dst = reinterpret_cast<float *>(h->ws + h->L.pops2);   // the lattice holding state t
    else p.dst = p.src;
    cudaError_t e;
    switch (h->V) {
    case 4: e = launch_setstate_v<4>(h, p, in_dev, odd); break;
    case 2: e = launch_setstate_v<2>(h, p, in_dev, odd); break;
    default: e = launch_setstate_v<1>(h, p, in_dev, odd); break;
    }
    CU_TRY(e);
    h->t = t; h->inited = true;
    return LBM_OK;
}

int lbm_stats_accumulate(lbm_t *h, int every)
{
    if (!h) return fail(LBM_EINVAL, "handle is NULL");
    if (every < 0) return fail(LBM_EINVAL, "every must be >= 0");
    h->stats_every = every; h->stats_phase = 0;
    return LBM_OK;
}

int lbm_stats_reset(lbm_t *h)
{
    if (!h) return fail(LBM_EINVAL, "handle is NULL");
    DevGuard dg(h);
    if (!h->bound) return fail(LBM_ESTATE, "lbm_stats_reset before lbm_bind");
    return stats_reset_impl(h);
}

int lbm_stats_read(lbm_t *h, double *out, long long *nsamples)
{
    if (!h) return fail(LBM_EINVAL, "handle is NULL");
    DevGuard dg(h);
    if (!h->bound) return fail(LBM_ESTATE, "lbm_stats_read before lbm_bind");
    if (!out) return fail(LBM_EINVAL, "out is NULL");
    // the running sums, the accumulation centres and the divergence flag lie next to one another in
    // the workspace: ONE device-to-host copy into a pinned mirror (three copies into pageable memory
    // cost 0.4 ms per call, 3 % of a cfg5 step in the end-to-end loop)
    CU_TRY(cudaMemcpyAsync(h->hpin, h->ws + h->L.acc, h->L.flag + 4 - h->L.acc, cudaMemcpyDeviceToHost, h->stream));
    CU_TRY(cudaStreamSynchronize(h->stream));
    const double *acc = reinterpret_cast<const double *>(h->hpin);
    const float *shift = reinterpret_cast<const float *>(h->hpin + (h->L.shift - h->L.acc));
    int flag;
    memcpy(&flag, h->hpin + (h->L.flag - h->L.acc), 4);
    if (nsamples) *nsamples = h->nsamples;
    const double cnt = (double)h->nsamples * h->nx * (h->zhi - h->zlo);
    for (int y = 0; y < h->ny; ++y) {
        const double *a = acc + (size_t)y * NSTAT;
        double *r = out + (size_t)y * NSTAT;
        if (h->nsamples == 0) { for (int k = 0; k < NSTAT; ++k) r[k] = 0.0; continue; }
        // sums are of (u - u0, v - v0, w - w0, rho - 1): second moments about the mean are
        // shift-invariant, first moments get the centre added back (R18)
        const double mu = a[0] / cnt, mv = a[1] / cnt, mw = a[2] / cnt;
        r[0] = mu + shift[y * 4 + 0]; r[1] = mv + shift[y * 4 + 1]; r[2] = mw + shift[y * 4 + 2];
        r[3] = a[3] / cnt - mu * mu; r[4] = a[4] / cnt - mv * mv; r[5] = a[5] / cnt - mw * mw;
        r[6] = a[6] / cnt - mu * mv; r[7] = a[7] / cnt - mv * mw; r[8] = a[8] / cnt - mu * mw;
        r[9] = (a[9] + (double)h->nsamples * h->nfluid[y]) / cnt;   // sum of rho = sum(rho-1) + fluid cells
    }
    if (flag) return fail(LBM_EDIVERGED, "non-finite plane sum of rho seen by the statistics reduction");
    return LBM_OK;
}

long long lbm_time(const lbm_t *h) { return h ? h->t : -1; }
long long lbm_launch_count(const lbm_t *h) { return h ? h->launches : -1; }
const char *lbm_variant(const lbm_t *h) { return h ? h->variant : ""; }

int lbm_set_kernel_timing(lbm_t *h, int on)
{
    if (!h) return fail(LBM_EINVAL, "handle is NULL");
    h->timing = on != 0;
    return LBM_OK;
}

int lbm_kernel_timing_read(lbm_t *h, double *total_ms, long long *launches)
{
    if (!h) return fail(LBM_EINVAL, "handle is NULL");
    DevGuard dg(h);
    if (!h->bound) return fail(LBM_ESTATE, "lbm_kernel_timing_read before lbm_bind");
    CU_TRY(cudaStreamSynchronize(h->stream));
    double tot = 0.0;
    for (size_t q = 0; q + 1 < h->ev_used; q += 2) {
        float ms = 0.f;
        CU_TRY(cudaEventElapsedTime(&ms, h->ev[q], h->ev[q + 1]));
        tot += ms;
    }
    if (total_ms) *total_ms = tot;
    if (launches) *launches = (long long)(h->ev_used / 2);
    h->ev_used = 0;
    return LBM_OK;
}

void lbm_destroy(lbm_t *h)
{
    if (!h) return;
    {
        DevGuard dg(h);
        graph_drop(h);
        for (cudaEvent_t e : h->ev) cudaEventDestroy(e);
        h->ev.clear();
        if (h->hpin) cudaFreeHost(h->hpin);
    }
    delete h;
}

int lbm_lad_profile(int hc, int ny, double LAI, double eta_m, double *out)
{
    if (!out || ny < 1 || hc < 0 || hc > ny) return fail(LBM_EINVAL, "bad lad_profile arguments");
    if (!(eta_m > 0.0 && eta_m < 1.0)) return fail(LBM_EINVAL, "eta_m must be in (0,1)");
    double sum = 0.0;
    for (int j = 0; j < ny; ++j) {
        double s = 0.0;
        if (j < hc) {
            // Eq. 14 (L107) with Eq. 15 (L112): n = 6 below the LAD maximum, 1/2 above
            const double eta = (j + 0.5) / hc;
            const double ratio = (1.0 - eta_m) / (1.0 - eta);
            const double n = (eta < eta_m) ? 6.0 : 0.5;
            s = std::exp(n * std::log(ratio) + n * (1.0 - ratio));
        }
        out[j] = s; sum += s;
    }
    for (int j = 0; j < ny; ++j) out[j] = (sum > 0.0) ? out[j] * (LAI / sum) : 0.0;
    return LBM_OK;
}

int lbm_lad_eq14(int hc, int ny, double a_fm, double eta_m, double *out)
{
    if (!out || ny < 1 || hc < 0 || hc > ny) return fail(LBM_EINVAL, "bad lad_eq14 arguments");
    if (!(a_fm >= 0.0) || !std::isfinite(a_fm)) return fail(LBM_EINVAL, "a_fm must be >= 0");
    if (!(eta_m >= 0.0 && eta_m < 1.0)) return fail(LBM_EINVAL, "eta_m must be in [0,1)");
    for (int j = 0; j < ny; ++j) {
        double a = 0.0;
        if (j < hc) {
            if (eta_m == 0.0) a = a_fm;               // constant LAD (Table II case 1)
            else {
                // Eq. 14 (L107) with Eq. 15 (L112), a_fm as printed (Table II case 2: 0.38 per metre)
                const double eta = (j + 0.5) / hc;
                const double ratio = (1.0 - eta_m) / (1.0 - eta);
                const double n = (eta < eta_m) ? 6.0 : 0.5;
                a = a_fm * std::exp(n * std::log(ratio) + n * (1.0 - ratio));
            }
        }
        out[j] = a;
    }
    return LBM_OK;
}

int lbm_wall_friction_velocity(double F, double H, double rho, double *u_tau)
{
    if (!u_tau) return fail(LBM_EINVAL, "u_tau is NULL");
    if (!(F >= 0.0) || !(H > 0.0) || !(rho > 0.0)) return fail(LBM_EINVAL, "need F >= 0, H > 0, rho > 0");
    *u_tau = std::sqrt(F * H / rho);   // Eq. 16 (L179): F = rho u_tau^2 / H
    return LBM_OK;
}

int lbm_forest_friction_velocity(const double *stats, int ny, int hc, double *u_star)
{
    if (!stats || !u_star) return fail(LBM_EINVAL, "NULL argument");
    if (hc < 1 || 2 * hc >= ny) return fail(LBM_EINVAL, "need 1 <= h and 2h < ny (h=%d, ny=%d)", hc, ny);
    const double *lo = stats + (size_t)(2 * hc - 1) * LBM_NSTAT, *hi = stats + (size_t)(2 * hc) * LBM_NSTAT;
    const double uv = 0.5 * (lo[6] + hi[6]), vw = 0.5 * (lo[7] + hi[7]);
    *u_star = std::sqrt(std::sqrt(uv * uv + vw * vw));   // L210
    return LBM_OK;
}

int lbm_stats_normalise(const double *stats, int ny, double u_ref, double *out)
{
    if (!stats || !out || ny < 1) return fail(LBM_EINVAL, "bad arguments");
    if (!(u_ref > 0.0)) return fail(LBM_EINVAL, "u_ref must be > 0");
    for (int j = 0; j < ny; ++j) {
        const double *a = stats + (size_t)j * LBM_NSTAT;
        double *r = out + (size_t)j * LBM_NSTAT;
        for (int k = 0; k < 3; ++k) r[k] = a[k] / u_ref;
        for (int k = 3; k < 6; ++k) r[k] = std::sqrt(a[k] > 0.0 ? a[k] : 0.0) / u_ref;
        for (int k = 6; k < 9; ++k) r[k] = a[k] / (u_ref * u_ref);
        r[9] = a[9];
    }
    return LBM_OK;
}

int lbm_wall_units(int ny, double u_tau, double nu, double *yplus)
{
    if (!yplus || ny < 1 || !(nu > 0.0) || !(u_tau >= 0.0)) return fail(LBM_EINVAL, "bad arguments");
    for (int j = 0; j < ny; ++j) yplus[j] = (j + 0.5) * u_tau / nu;
    return LBM_OK;
}

uint64_t lbm_mix64(uint64_t seed, uint64_t ctr) { return lbm::mix64(seed, ctr); }

