// lbm_kernels.cuh — sm_100a kernels of the fused D3Q19 LES + forest-canopy LBM step.
//
// One kernel launch = one time step of Algorithm 1: stream (Eq. 1),
// moments (Eqs. 5-7), predictor velocity + forest drag + velocity correction (Eq. 6,
// Eq. 13, Alg. 1), Smagorinsky tau_total (Eqs. 10-12), Guo-forced BGK
// collision (Eqs. 1-4), boundary links (L177, L216) and the store, with the stage-1
// x-row sums of the plane statistics (L200, L251) fused into the epilogue.
//
// B200 design: HBM-bound stencil, 152 B per cell update.
//  * populations are fp32 structure-of-arrays, stored SHIFTED (g_i = f_i - w_i) so that fp32
//    rounding acts on the O(Ma) deviation instead of on the O(1) weights;
//  * each thread owns V = 4 (2, 1) consecutive x cells: every population row is moved with
//    aligned 128-bit (64-, 32-bit) loads and stores; the +-1 x shift of 10 of the 19 directions
//    is done in registers with one warp shuffle, only the two edge lanes of a warp touch one
//    extra element;
//  * two storage schemes: two-lattice pull (src -> dst) and the in-place AA pattern (even step
//    reads/writes its own cell with swapped slots, odd step reads/writes the neighbours), which
//    halves the memory and makes config 5 (604 M cells) a 46 GB problem;
//  * boundary rows are handled by per-lane slot/row selection (no divergent shuffles), flags are
//    a handful of bits in a kernel parameter, the canopy is a per-row table (C_D a_j).
//
// This file shares nothing with oracle/ (different arithmetic form: pairwise even/odd
// collision on shifted populations, fp32).
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>
#include <type_traits>

namespace lbm {

constexpr int Q = 19;
constexpr int NSTAT = 10;
constexpr int MAX_THREADS = 256;

// D3Q19 velocity set in the specification numbering (include/lbm.h).
struct Lat {
    static constexpr int cx[Q] = {0, 1, -1, 0, 0, 0, 0, 1, -1, 1, -1, 1, -1, 1, -1, 0, 0, 0, 0};
    static constexpr int cy[Q] = {0, 0, 0, 1, -1, 0, 0, 1, -1, -1, 1, 0, 0, 0, 0, 1, -1, 1, -1};
    static constexpr int cz[Q] = {0, 0, 0, 0, 0, 1, -1, 0, 0, 0, 0, 1, -1, -1, 1, 1, -1, -1, 1};
    static constexpr int opp[Q] = {0, 2, 1, 4, 3, 6, 5, 8, 7, 10, 9, 12, 11, 14, 13, 16, 15, 18, 17};
    static constexpr int mir[Q] = {0, 1, 2, 4, 3, 5, 6, 9, 10, 7, 8, 11, 12, 13, 14, 18, 17, 16, 15};
};

// How the streamed (pre-collision) populations of a cell are fetched / how the post-collision
// ones are put back.
enum ReadMode { RD_LOCAL = 0,    // A[i][x]                         (AA even step; AA state, t even)
                RD_PULL = 1,     // A[i][x - c_i]                   (two-lattice)
                RD_PULL_OPP = 2, // A[opp i][x - c_i]               (AA odd step; AA state, t odd)
                RD_XE = 3,       // x-balanced AA, even step        (see below)
                RD_XO = 4        // x-balanced AA, odd step
};
enum WriteMode { WR_LOCAL = 0,     // B[i][x]                      (two-lattice)
                 WR_LOCAL_OPP = 1, // A[opp i][x]                  (AA even step)
                 WR_PUSH = 2,      // A[i][x + c_i]                (AA odd step, AA init)
                 WR_XE = 3,        // x-balanced AA, even step
                 WR_XO = 4         // x-balanced AA, odd step
};
// x-balanced AA ("AAX").  In the AA pattern the even step touches only its own cell and the odd
// step does all the streaming: 10 x-shifted reads and 10 x-shifted writes, which on 128-bit
// accesses cost shuffles and scalar edge accesses, so the odd step is issue-bound where the even
// one is bandwidth-bound.  Any in-place scheme is hazard-free as long as every cell writes exactly
// the locations it read; that leaves the freedom to keep the x part of the displacement of some
// populations for the other step.  With a_i = 1 for c_ix = +1 (else 0), population i of cell x
// lives at slot i, cell x + c_i - a_i e_x after an odd step and at slot opp(i), cell x - a_opp(i) e_x
// after an even step.  Net effect, identical in BOTH steps and independent of wall / free-slip
// redirections (which only change slot and row, as in AA): populations with c_x = +1 are READ from
// x - 1, populations with c_x = -1 are WRITTEN to x - 1, nothing else moves in x.  Each step then
// has 5 x-shifted reads and 5 x-shifted writes; rows (y, z) and slots follow AA exactly.

enum { BC_BOT_WALL = 0, BC_BOT_PERIODIC = 1 };
enum { BC_TOP_WALL = 0, BC_TOP_SLIP = 1, BC_TOP_PERIODIC = 2, BC_TOP_LID = 3 };

struct KParams {
    float *src;          // population array read  [19][N]
    float *dst;          // population array written (== src for AA)
    int nx, ny, nz;
    int nchunk;          // blocks per x row
    int pchunks;         // x chunks per row in the layout of `partial` (>= nchunk of any kernel in use)
    int wpart;           // 1 = every warp of a row segment stores its own partial (no block-level reduce;
                         //     pchunks = nchunk * warps per segment): geometry handles, where one warp of a
                         //     block may take the slow geometry path and the others should not wait for it
    long long N;
    // physics (fp32 copies)
    float tau0, tau0sq, ksmag;  // ksmag = 18 sqrt(2) Cs^2
    float Fbx, Fby, Fbz;        // body force density F_b
    const float *cda;           // [ny] C_D * a_j   (0 = not forest)
    const float2 *sgs;          // [ny] per-row SGS table {tau0 - 3 C_j Sbar_j, 18 sqrt(2) C_j}; NULL = the
                                // standard Smagorinsky model with the constants above (lbm_set_sgs_rows)
    const float *jref;          // [ny] r_j = J0_j / 12: per-row momentum reference (see mom_ref_shift)
    int bot, top, drag_vector;
    int aax;                    // 1 = x-balanced AA storage (host-side kernels that address single entries)
    const unsigned *solid;      // per-cell solid bit mask, one word per 32 x cells (NULL = none)
    const unsigned *solid_nb;   // the same mask dilated by one cell in x, y, z (host-built)
    int nxw;                    // words per x row, ceil(nx / 32) (bits past nx in the last word are 0)
    const unsigned char *fidx;  // per-cell forest table index (0 = none), NULL = no coded forest
    const float *ftab;          // [256] C_D * a_f of the forest codes in use
    const unsigned char *frow;  // [ny] 1 = the row holds coded forest cells
    const unsigned char *bflag; // per thread block of the step launch: 1 = geometry (a solid cell within one
                                // step of the block's cells, or a coded forest cell), 0 = plain fluid
    float lid[5];               // forced-equilibrium lid: f_eq,i(1, U_top) - w_i for i = 4, 8, 9, 16, 18
    // statistics
    float *partial;             // [ny][NSTAT][nz*nchunk]
    const float *shift;         // [ny][4] accumulation centre (u0, v0, w0, -), may be NULL
    // macros / init
    float *rho_out, *u_out;
    int *diverged;              // set to 1 by macros_kernel when it sees a non-finite density
    const float *rho_in, *u_in; // init from fields (NULL -> synthetic)
    const float *uprof;         // [ny] synthetic profile U(y_j)
    double noise_amp;           // noise_frac * U_ref
    unsigned long long seed;
    int z0, z1;                 // z range of a launch (chunked host transfers; interior planes of a slab)
    int rev;                    // 1 = the blocks walk the rows of the launch from the last to the first
    int grid3;                  // 1 = 3-D grid (x chunk, row block of a plane, plane): the step launch when the
                                //     block rows divide ny - no integer division in the index arithmetic
    int zg0, nzg;               // z slab: global z of local plane 0 and global nz (init recipe only)
    int zv0, zv1;               // planes that hold the lattice proper ([1, nz-1) on a z slab: not the ghosts)
    long long zoff;             // element offset of plane z0 inside rho_in/u_in/rho_out/u_out
    long long Nio;              // component stride of u_in / u_out
};

// ---------------------------------------------------------------------------------------------
// small helpers
// ---------------------------------------------------------------------------------------------
template <int I, int N, class F>
__device__ __forceinline__ void static_for(F &&f)
{
    if constexpr (I < N) {
        f(std::integral_constant<int, I>{});
        static_for<I + 1, N>(f);
    }
}

// LBM_CS (build-time experiment switch, default 0): bit 0 = population loads with the streaming
// cache hint (ld.global.cs), bit 1 = population stores with it (st.global.cs).
#ifndef LBM_CS
#define LBM_CS 0
#endif
template <int V> __device__ __forceinline__ void ldv(const float *p, float (&o)[V])
{
    if constexpr (V == 4) {
#if LBM_CS & 1
        float4 t = __ldcs(reinterpret_cast<const float4 *>(p));
#else
        float4 t = *reinterpret_cast<const float4 *>(p);
#endif
        o[0] = t.x; o[1] = t.y; o[2] = t.z; o[3] = t.w;
    } else if constexpr (V == 2) {
        float2 t = *reinterpret_cast<const float2 *>(p);
        o[0] = t.x; o[1] = t.y;
    } else {
        o[0] = *p;
    }
}
template <int V> __device__ __forceinline__ void stv(float *p, const float (&o)[V])
{
#if LBM_CS & 2
    if constexpr (V == 4) __stcs(reinterpret_cast<float4 *>(p), make_float4(o[0], o[1], o[2], o[3]));
#else
    if constexpr (V == 4) *reinterpret_cast<float4 *>(p) = make_float4(o[0], o[1], o[2], o[3]);
#endif
    else if constexpr (V == 2) *reinterpret_cast<float2 *>(p) = make_float2(o[0], o[1]);
    else *p = o[0];
}

// Per-thread geometry: V cells x0..x0+V-1 of row (y, z).
struct Ctx {
    int x0, y, z, chunk;
    int xl, xr;        // wrapped x0-1, x0+V
    int ym, yp, zm, zp; // neighbour rows (wrapped / clamped)
    bool bot_bb, top_bb, top_fs, top_lid; // this row touches a wall / free-slip / lid face
    bool edgeL, edgeR;  // lane has no x-neighbour lane on that side
};

// Sweep direction.  Blocks are scheduled in index order, so the rows a launch touches last are the
// ones the 126 MB L2 still holds when the next launch starts.  Consecutive time steps walk the
// lattice in opposite directions (p.rev alternates): a step starts on the planes the previous one
// has just written and takes them from L2 instead of DRAM.  The order of the blocks has no effect
// on the result (two-lattice: src and dst differ; in place: a block writes exactly what it read).
__device__ __forceinline__ int block_index(const KParams &p)
{
    return p.rev ? (int)(gridDim.x - 1u - blockIdx.x) : (int)blockIdx.x;
}
// The same block order on a 3-D grid (blocks are dispatched x fastest, then y, then z): x = chunk of
// the row, y = row block inside the plane, z = plane of the launch.  Saves the two integer divisions
// (block -> row, row -> plane) of the 1-D form: ~55 of ~1450 instructions per thread.
__device__ __forceinline__ void block_index3(const KParams &p, int &cb, int &yb, int &zb)
{
    cb = (int)blockIdx.x; yb = (int)blockIdx.y; zb = (int)blockIdx.z;
    if (p.rev) { cb = (int)gridDim.x - 1 - cb; yb = (int)gridDim.y - 1 - yb; zb = (int)gridDim.z - 1 - zb; }
}
// index of the block in the whole-lattice order of the 1-D launch (per-block geometry flags)
__device__ __forceinline__ long long block_linear(const KParams &p)
{
    if (p.grid3) {
        // gridDim.y is the number of row blocks of a plane: no division on this path
        int cb, yb, zb;
        block_index3(p, cb, yb, zb);
        return ((long long)(p.z0 + zb) * (int)gridDim.y + yb) * p.nchunk + cb;
    }
    return (long long)block_index(p) + (long long)(p.z0 * p.ny / (int)blockDim.y) * p.nchunk;
}

// Programmatic dependent launch (lbm_launch.cuh: launch_chain): wait until the preceding launch of the
// chain has completed and its writes are visible, then let the following launch be set up.  Both are
// no-ops for a kernel that was launched without the attribute.  Must run before the first access to
// anything a preceding kernel wrote.
__device__ __forceinline__ void pdl_enter()
{
    asm volatile("griddepcontrol.wait;" ::: "memory");
    asm volatile("griddepcontrol.launch_dependents;" ::: "memory");
}

// `again`: recompute from laundered thread/block indices, so that the compiler does not keep the
// first Ctx alive across the collision (register pressure of the AA odd step).
// (A variant for launches with blockDim.y == 1 that drops threadIdx.y, so that the row and everything
// derived from it becomes block-uniform and moves to the uniform datapath, was measured on cfg5: 7 %
// fewer per-thread instructions, SM clock under the power cap 1635 instead of 1575 MHz, and 3.6 %
// SLOWER - 40.1 against 41.6 GLUPS; the uniform pipe is the slower one.  Dropped.)
template <int V> __device__ __forceinline__ Ctx make_ctx(const KParams &p, int row0, bool again = false)
{
    Ctx c;
    int tx = threadIdx.x, ty = threadIdx.y;
    if (p.grid3) {
        int cb, yb, zb;
        block_index3(p, cb, yb, zb);
        if (again) asm volatile("" : "+r"(tx), "+r"(ty), "+r"(cb), "+r"(yb), "+r"(zb));
        c.chunk = cb;
        c.y = yb * (int)blockDim.y + ty;
        c.z = p.z0 + zb;
    } else {
        int bx = block_index(p);
        if (again) asm volatile("" : "+r"(tx), "+r"(ty), "+r"(bx));
        // 1-D grid, the x chunks of a row are consecutive blocks (they run together, so the partial
        // sectors at the chunk seams of the shifted stores merge in L2)
        const int rb = bx / p.nchunk;
        c.chunk = bx - rb * p.nchunk;
        const int row = row0 + rb * blockDim.y + ty;
        c.z = row / p.ny;
        c.y = row - c.z * p.ny;
    }
    const int lane = (ty * blockDim.x + tx) & 31;
    c.x0 = (c.chunk * blockDim.x + tx) * V;
    c.xl = (c.x0 == 0) ? p.nx - 1 : c.x0 - 1;
    c.xr = (c.x0 + V >= p.nx) ? 0 : c.x0 + V;
    c.zm = (c.z == 0) ? p.nz - 1 : c.z - 1;
    c.zp = (c.z == p.nz - 1) ? 0 : c.z + 1;
    const bool isbot = (c.y == 0), istop = (c.y == p.ny - 1);
    c.ym = isbot ? (p.bot == BC_BOT_PERIODIC ? p.ny - 1 : c.y) : c.y - 1;
    c.yp = istop ? (p.top == BC_TOP_PERIODIC ? 0 : c.y) : c.y + 1;
    c.bot_bb = isbot && p.bot == BC_BOT_WALL;
    // the lid face addresses like a wall (own cell, opposite slot); loads then take the lid value
    c.top_lid = istop && p.top == BC_TOP_LID;
    c.top_bb = istop && (p.top == BC_TOP_WALL || p.top == BC_TOP_LID);
    c.top_fs = istop && p.top == BC_TOP_SLIP;
    c.edgeL = (lane == 0) || (tx == 0);
    c.edgeR = (lane == 31) || (tx == (int)blockDim.x - 1);
    return c;
}

// ---------------------------------------------------------------------------------------------
// S1: stream.  Fetch the V incoming populations of direction I (Eq. 1 LHS, L41; Alg. 1).
//   normal link      : slot I      at (x - c_x, y - c_y, z - c_z), periodic wrap in x, z (L177)
//   wall face        : slot opp(I) at the cell itself (halfway bounce-back; R11, R12)
//   free-slip face   : slot mir(I) at (x - c_x, y, z - c_z)  (specular reflection; R13)
// RD_PULL_OPP stores every population in the opposite slot (AA after an even step).
// ---------------------------------------------------------------------------------------------
template <int V, int RM, int I>
__device__ __forceinline__ void load_dir(const KParams &p, const Ctx &c, float (&o)[V])
{
    constexpr int cx = Lat::cx[I], cy = Lat::cy[I], cz = Lat::cz[I];
    if constexpr (RM == RD_LOCAL) {
        ldv<V>(p.src + (long long)I * p.N + ((long long)(c.y + p.ny * c.z) * p.nx + c.x0), o);
        return;
    } else {
        constexpr bool AAX = (RM == RD_XE || RM == RD_XO);
        // the fetch comes from x - XS; the classic modes cancel the shift on a bounce-back link
        constexpr int XS = AAX ? (cx == 1 ? 1 : 0) : cx;
        bool bb = false, fs = false;
        const float *rowp;
        if constexpr (RM == RD_XE) {
            rowp = p.src + (long long)I * p.N + (long long)(c.y + p.ny * c.z) * p.nx;
        } else {
            constexpr int S_N = (RM == RD_PULL) ? I : Lat::opp[I];
            constexpr int S_BB = (RM == RD_PULL) ? Lat::opp[I] : I;
            constexpr int S_FS = (RM == RD_PULL) ? Lat::mir[I] : Lat::opp[Lat::mir[I]];
            if constexpr (cy == 1) bb = c.bot_bb;
            if constexpr (cy == -1) { bb = c.top_bb; fs = c.top_fs; }
            const int ysel = (cy == 0) ? c.y : (cy == 1 ? c.ym : c.yp);
            const int zsel = (cz == 0) ? c.z : (cz == 1 ? c.zm : c.zp);
            const int slot = bb ? S_BB : (fs ? S_FS : S_N);
            const int yrow = (bb || fs) ? c.y : ysel;
            const int zrow = bb ? c.z : zsel;
            rowp = p.src + (long long)slot * p.N + (long long)(yrow + p.ny * zrow) * p.nx;
        }
        const bool cancel = AAX ? false : bb;
        if constexpr (XS == 0) {
            ldv<V>(rowp + c.x0, o);
        } else if constexpr (V == 1) {
            const int xs = cancel ? c.x0 : (XS == 1 ? c.xl : c.xr);
            o[0] = rowp[xs];
        } else {
            float v[V];
            ldv<V>(rowp + c.x0, v);
            if constexpr (XS == 1) {           // need x0-1 .. x0+V-2
                const bool need = c.edgeL && !cancel;
                float e = 0.f;
                if (need) e = rowp[c.xl];
                float l = __shfl_up_sync(0xffffffffu, v[V - 1], 1);
                l = c.edgeL ? e : l;
                o[0] = cancel ? v[0] : l;
#pragma unroll
                for (int k = 1; k < V; ++k) o[k] = cancel ? v[k] : v[k - 1];
            } else {                            // need x0+1 .. x0+V
                const bool need = c.edgeR && !cancel;
                float e = 0.f;
                if (need) e = rowp[c.xr];
                float r = __shfl_down_sync(0xffffffffu, v[0], 1);
                r = c.edgeR ? e : r;
#pragma unroll
                for (int k = 0; k < V - 1; ++k) o[k] = cancel ? v[k] : v[k + 1];
                o[V - 1] = cancel ? v[V - 1] : r;
            }
        }
    }
}

// ---------------------------------------------------------------------------------------------
// S7: store the V post-collision populations of direction I.
//   WR_LOCAL / WR_LOCAL_OPP : own cell, slot I / opp(I), aligned.
//   WR_PUSH (AA odd step)   : slot I at (x + c); a link that leaves through a wall face goes to
//                             slot opp(I) of the own cell, through a free-slip face to slot
//                             mir(I) at (x + c_x, y, z + c_z) - the places where the next even
//                             step expects its incoming populations.
// ---------------------------------------------------------------------------------------------
// `act` = false: the lane takes part in the shuffles but stores nothing (solid-mask slow path).
template <int V, int WM, int I>
__device__ __forceinline__ void store_dir(const KParams &p, const Ctx &c, const float (&r)[V], bool act = true)
{
    constexpr int cx = Lat::cx[I], cy = Lat::cy[I], cz = Lat::cz[I];
    if constexpr (WM == WR_LOCAL || WM == WR_LOCAL_OPP) {
        constexpr int S = (WM == WR_LOCAL) ? I : Lat::opp[I];
        stv<V>(p.dst + (long long)S * p.N + ((long long)(c.y + p.ny * c.z) * p.nx + c.x0), r);
        return;
    } else {
        constexpr bool AAX = (WM == WR_XE || WM == WR_XO);
        // the values land on x + XS; the classic push cancels the shift on a bounce-back link
        constexpr int XS = AAX ? (cx == -1 ? -1 : 0) : cx;
        bool bb = false, fs = false;
        float *rowp;
        if constexpr (WM == WR_XE) {
            rowp = p.dst + (long long)Lat::opp[I] * p.N + (long long)(c.y + p.ny * c.z) * p.nx;
        } else {
            if constexpr (cy == -1) bb = c.bot_bb;
            if constexpr (cy == 1) { bb = c.top_bb; fs = c.top_fs; }
            const int ysel = (cy == 0) ? c.y : (cy == 1 ? c.yp : c.ym);
            const int zsel = (cz == 0) ? c.z : (cz == 1 ? c.zp : c.zm);
            constexpr int S_BB = Lat::opp[I], S_FS = Lat::mir[I];
            const int slot = bb ? S_BB : (fs ? S_FS : I);
            const int yrow = (bb || fs) ? c.y : ysel;
            const int zrow = bb ? c.z : zsel;
            rowp = p.dst + (long long)slot * p.N + (long long)(yrow + p.ny * zrow) * p.nx;
        }
        const bool cancel = AAX ? false : bb;
        if constexpr (XS == 0) {
            if (act) stv<V>(rowp + c.x0, r);
        } else if constexpr (V == 1) {
            const int xs = cancel ? c.x0 : (XS == 1 ? c.xr : c.xl);
            if (act) rowp[xs] = r[0];
        } else {
            if constexpr (XS == 1) {           // values land on x0+1 .. x0+V
                const float l = __shfl_up_sync(0xffffffffu, r[V - 1], 1);
                if (!act) {
                } else if (cancel) {
                    stv<V>(rowp + c.x0, r);
                } else {
                    if (!c.edgeL) {
                        float t[V];
                        t[0] = l;
#pragma unroll
                        for (int k = 1; k < V; ++k) t[k] = r[k - 1];
                        stv<V>(rowp + c.x0, t);
                    } else if constexpr (V == 4) {     // x0+1 alone, then the 8-byte aligned pair x0+2, x0+3
                        rowp[c.x0 + 1] = r[0];
                        *reinterpret_cast<float2 *>(rowp + c.x0 + 2) = make_float2(r[1], r[2]);
                    } else {
#pragma unroll
                        for (int k = 0; k < V - 1; ++k) rowp[c.x0 + 1 + k] = r[k];
                    }
                    if (c.edgeR) rowp[c.xr] = r[V - 1];
                }
            } else {                            // values land on x0-1 .. x0+V-2
                const float rr = __shfl_down_sync(0xffffffffu, r[0], 1);
                if (!act) {
                } else if (cancel) {
                    stv<V>(rowp + c.x0, r);
                } else {
                    if (!c.edgeR) {
                        float t[V];
#pragma unroll
                        for (int k = 0; k < V - 1; ++k) t[k] = r[k + 1];
                        t[V - 1] = rr;
                        stv<V>(rowp + c.x0, t);
                    } else if constexpr (V == 4) {     // the 8-byte aligned pair x0, x0+1, then x0+2 alone
                        *reinterpret_cast<float2 *>(rowp + c.x0) = make_float2(r[1], r[2]);
                        rowp[c.x0 + 2] = r[3];
                    } else {
#pragma unroll
                        for (int k = 1; k < V; ++k) rowp[c.x0 + k - 1] = r[k];
                    }
                    if (c.edgeL) rowp[c.xl] = r[0];
                }
            }
        }
    }
}

// Forced-equilibrium top ("the top boundary is forced to be in equilibrium with the
// same velocity as the free-stream flow"): the populations that enter
// through the top face are f_eq,i(1, U_top), whatever the storage holds there.
__host__ __device__ constexpr int lid_index(int i)
{
    return i == 4 ? 0 : i == 8 ? 1 : i == 9 ? 2 : i == 16 ? 3 : i == 18 ? 4 : -1;
}

// ---------------------------------------------------------------------------------------------
// Per-cell solid mask (PAPER.md:L129-135 bit-coded geometry, L226 trip boxes; SURVEY.md §8(f)
// NEXT #2).  One bit per cell, word = 32 consecutive x cells of a row.  A link whose other end is
// a solid cell is a halfway bounce-back link, exactly like a wall face; solid cells themselves
// keep the rest state (g = 0) and are never updated.
//
// A thread gathers, for each of the 9 (y, z) rows its links touch, the V+2 bits of the cells
// x0-1 .. x0+V into 6-bit fields packed in one 64-bit word: field (a, b), a in {ym, y, yp},
// b in {zm, z, zp}, at bit 6*(3a + b); bit 0 = cell x0-1, bit k+1 = cell x0+k.
// ---------------------------------------------------------------------------------------------
template <int V>
__device__ __forceinline__ unsigned solid_field(const KParams &p, const Ctx &c, int yrow, int zrow)
{
    const unsigned *row = p.solid + (long long)(yrow + p.ny * zrow) * p.nxw;
    const int w = c.x0 >> 5, b = c.x0 & 31;
    const unsigned m = __ldg(row + w);
    unsigned f = ((m >> b) & ((1u << V) - 1u)) << 1;
    // left neighbour x0-1 (periodic: x = nx-1 sits at bit (nx-1)&31 of the last word)
    if (c.x0 == 0) f |= (__ldg(row + p.nxw - 1) >> ((p.nx - 1) & 31)) & 1u;
    else if (b > 0) f |= (m >> (b - 1)) & 1u;
    else f |= __ldg(row + w - 1) >> 31;
    // right neighbour x0+V (periodic: x = 0)
    if (c.x0 + V >= p.nx) f |= (__ldg(row) & 1u) << (V + 1);
    else if (b + V < 32) f |= ((m >> (b + V)) & 1u) << (V + 1);
    else f |= (__ldg(row + w + 1) & 1u) << (V + 1);
    return f;
}

// one word of the dilated mask tells whether any cell within one step of the own cells is solid
__device__ __forceinline__ unsigned solid_nb_word(const KParams &p, const Ctx &c)
{
    return __ldg(p.solid_nb + (long long)(c.y + p.ny * c.z) * p.nxw + (c.x0 >> 5));
}

template <int V>
__device__ __forceinline__ unsigned long long solid_gather_rows(const KParams &p, const Ctx &c)
{
    const int ys[3] = {c.ym, c.y, c.yp}, zs[3] = {c.zm, c.z, c.zp};
    unsigned long long S = 0ull;
#pragma unroll
    for (int a = 0; a < 3; ++a)
#pragma unroll
        for (int b = 0; b < 3; ++b)
            S |= (unsigned long long)solid_field<V>(p, c, ys[a], zs[b]) << (6 * (3 * a + b));
    return S;
}
template <int V>
__device__ __forceinline__ unsigned long long solid_gather(const KParams &p, const Ctx &c, unsigned nb)
{
    // if no cell within one step is solid every field is zero and the nine-row gather is skipped
    if (((nb >> (c.x0 & 31)) & ((1u << V) - 1u)) == 0u) return 0ull;
    const int ys[3] = {c.ym, c.y, c.yp}, zs[3] = {c.zm, c.z, c.zp};
    unsigned long long S = 0ull;
#pragma unroll
    for (int a = 0; a < 3; ++a)
#pragma unroll
        for (int b = 0; b < 3; ++b)
            S |= (unsigned long long)solid_field<V>(p, c, ys[a], zs[b]) << (6 * (3 * a + b));
    return S;
}
__device__ __forceinline__ unsigned solid_pick(unsigned long long S, int a, int b)
{
    return (unsigned)(S >> (6 * (3 * a + b))) & 63u;
}
// own cells of the thread: bit k = cell x0+k is solid
template <int V> __device__ __forceinline__ unsigned solid_self(unsigned long long S)
{
    return (solid_pick(S, 1, 1) >> 1) & ((1u << V) - 1u);
}

// C_D a_f of the thread's cells: the row table, overridden cell by cell where a forest code is set
// (Alg. 1 "if forest cell"; geometry handles only).  forest_idx fetches the
// V table indices of the thread's cells packed in one word (0 = no coded cell in the row).
template <int V, bool MASK>
__device__ __forceinline__ unsigned forest_idx(const KParams &p, const Ctx &c)
{
    unsigned idx = 0u;
    if constexpr (MASK) {
        if (p.fidx && __ldg(p.frow + c.y)) {
            const unsigned char *q = p.fidx + ((long long)(c.y + p.ny * c.z) * p.nx + c.x0);
            if constexpr (V == 4) idx = __ldg(reinterpret_cast<const unsigned *>(q));
            else if constexpr (V == 2) idx = __ldg(reinterpret_cast<const unsigned short *>(q));
            else idx = __ldg(q);
        }
    }
    return idx;
}
template <bool MASK>
__device__ __forceinline__ float cell_cda(const KParams &p, float row, unsigned idx, int k)
{
    if constexpr (MASK) {
        const unsigned t = (idx >> (8 * k)) & 255u;
        if (t) return __ldg(p.ftab + t);
    }
    return row;
}

template <int V, int RM>
__device__ __forceinline__ void load_all(const KParams &p, const Ctx &c, float (&g)[Q][V])
{
    static_for<0, Q>([&](auto ic) {
        constexpr int i = decltype(ic)::value;
        load_dir<V, RM, i>(p, c, g[i]);
        if constexpr (Lat::cy[i] == -1) {
            if (c.top_lid) {
#pragma unroll
                for (int k = 0; k < V; ++k) g[i][k] = p.lid[lid_index(i)];
            }
        }
    });
}

// Solid-mask correction of the streamed populations, applied after load_all (so that the 19
// loads do not wait for the mask): a link whose source cell (x0+k - c_x, in the row load_dir
// used) is solid bounces back, i.e. takes the own cell's opposite-slot value.
template <int V, int RM>
__device__ __forceinline__ void solid_fix_loads(const KParams &p, const Ctx &c, float (&g)[Q][V],
                                                unsigned long long S)
{
    // RD_LOCAL / RD_XE (the even steps of the single-array schemes): every population waits where the
    // odd step - which knows the geometry - has put it; nothing to correct.
    if constexpr (RM == RD_LOCAL || RM == RD_XE) return;
    // x-balanced AA, odd step: a bounce changes slot and row only, the x displacement of the fetch stays
    // (c_x = +1 populations come from x - 1 of the own row as well)
    constexpr bool AAX = (RM == RD_XO);
    // Which cells of direction i bounce: the bits of the source cells x0+k - c_x in the row load_dir used.
    auto bounce_bits = [&](auto ic) -> unsigned {
        constexpr int i = decltype(ic)::value;
        constexpr int cx = Lat::cx[i], cy = Lat::cy[i], cz = Lat::cz[i];
        bool bb = false, fs = false;
        if constexpr (cy == 1) bb = c.bot_bb;
        if constexpr (cy == -1) { bb = c.top_bb; fs = c.top_fs; }
        const int a = (bb || fs) ? 1 : 1 - cy, b = bb ? 1 : 1 - cz;
        return bb ? 0u : (solid_pick(S, a, b) >> (1 - cx)) & ((1u << V) - 1u);
    };
    // The own-cell loads of the bouncing links are issued in batches of six directions and consumed
    // afterwards: three dependent round trips to memory instead of up to eighteen.
    const float *ownp = p.src + ((long long)(c.y + p.ny * c.z) * p.nx + c.x0);
    static_for<0, 3>([&](auto bc) {
        constexpr int i0 = 1 + 6 * decltype(bc)::value;
        float own[6][V];
        unsigned bits[6];
        static_for<0, 6>([&](auto jc) {
            constexpr int j = decltype(jc)::value, i = i0 + j;
            constexpr int S_BB = (RM == RD_PULL) ? Lat::opp[i] : i;
            bits[j] = bounce_bits(std::integral_constant<int, i>{});
            if constexpr (AAX && Lat::cx[i] == 1) {
                const float *q = ownp + (long long)S_BB * p.N;
#pragma unroll
                for (int k = 0; k < V; ++k)
                    if ((bits[j] >> k) & 1u) own[j][k] = (k == 0) ? q[c.xl - c.x0] : q[k - 1];
            } else {
                if (bits[j]) ldv<V>(ownp + (long long)S_BB * p.N, own[j]);
            }
        });
        static_for<0, 6>([&](auto jc) {
            constexpr int j = decltype(jc)::value, i = i0 + j;
            if (bits[j]) {
#pragma unroll
                for (int k = 0; k < V; ++k)
                    if ((bits[j] >> k) & 1u) g[i][k] = own[j][k];
            }
        });
    });
}

template <int V, int WM, bool MASK>
__device__ __forceinline__ void store_all(const KParams &p, const Ctx &c, float (&g)[Q][V],
                                          unsigned long long S = 0ull)
{
    if constexpr (!MASK) {
        static_for<0, Q>([&](auto ic) {
            constexpr int i = decltype(ic)::value;
            store_dir<V, WM, i>(p, c, g[i]);
        });
    } else if constexpr (WM != WR_PUSH && WM != WR_XO) {
        const unsigned self = solid_self<V>(S);
        static_for<0, Q>([&](auto ic) {
            constexpr int i = decltype(ic)::value;
#pragma unroll
            for (int k = 0; k < V; ++k)
                if ((self >> k) & 1u) g[i][k] = 0.f;       // solid cells keep the rest state
            store_dir<V, WM, i>(p, c, g[i]);
        });
    } else {
        // WR_PUSH (AA) and WR_XO (x-balanced AA): the odd steps.  In the x-balanced pattern the values of
        // a c_x = -1 direction land one cell to the left and nothing else moves in x, whether the link
        // is open or bounces (a bounce changes slot and row only).
        constexpr bool AAX = (WM == WR_XO);
        const unsigned selff = solid_pick(S, 1, 1), self = solid_self<V>(S);
        const long long own = (long long)(c.y + p.ny * c.z) * p.nx + c.x0;
        static_for<0, Q>([&](auto ic) {
            constexpr int i = decltype(ic)::value;
            constexpr int cx = Lat::cx[i], cy = Lat::cy[i], cz = Lat::cz[i];
            constexpr int XS = AAX ? (cx == -1 ? -1 : 0) : cx;      // x displacement of the stored values
            bool bb = false, fs = false;
            if constexpr (cy == -1) bb = c.bot_bb;
            if constexpr (cy == 1) { bb = c.top_bb; fs = c.top_fs; }
            const int a = (bb || fs) ? 1 : 1 + cy, b = bb ? 1 : 1 + cz;
            const unsigned destf = bb ? 0u : solid_pick(S, a, b);
            // fast (vector) path only where neither the own cells, their x neighbours nor the
            // destination cells are solid
            const bool fast = (i == 0) ? (self == 0u) : ((selff | destf) == 0u);
            store_dir<V, WM, i>(p, c, g[i], fast);
            // the element a vector-path x neighbour expects THIS lane to store for it
            float nb = 0.f;
            if constexpr (V > 1 && XS == 1) nb = __shfl_up_sync(0xffffffffu, g[i][V - 1], 1);
            if constexpr (V > 1 && XS == -1) nb = __shfl_down_sync(0xffffffffu, g[i][0], 1);
            if (!fast) {
                const int ysel = (cy == 0) ? c.y : (cy == 1 ? c.yp : c.ym);
                const int zsel = (cz == 0) ? c.z : (cz == 1 ? c.zp : c.zm);
                constexpr int S_FS = Lat::mir[i], S_OPP = Lat::opp[i];
                const int slot = fs ? S_FS : i;
                const int yrow = fs ? c.y : ysel;
                float *rowp = p.dst + (long long)slot * p.N + (long long)(yrow + p.ny * zsel) * p.nx;
                float *ownp = p.dst + (long long)S_OPP * p.N + own;
                if constexpr (AAX) {
                    float *ownrow = ownp - c.x0;                          // slot opp(i), own row
#pragma unroll
                    for (int k = 0; k < V; ++k) {
                        if ((self >> k) & 1u) continue;                   // solid source: nothing leaves it
                        int xd = c.x0 + k + XS;
                        xd = (xd < 0) ? p.nx - 1 : xd;
                        const bool bounced = bb || ((destf >> (k + cx + 1)) & 1u);
                        (bounced ? ownrow : rowp)[xd] = g[i][k];
                    }
                    // the element a vector-path right neighbour expects THIS lane to store for it (its
                    // cell x0+V, landing on x0+V-1), bounced or not
                    if constexpr (V > 1 && XS == -1) {
                        if (!c.edgeR && !((selff >> (V + 1)) & 1u))
                            ((bb || ((destf >> V) & 1u)) ? ownrow : rowp)[c.x0 + V - 1] = nb;
                    }
                    return;
                }
#pragma unroll
                for (int k = 0; k < V; ++k) {
                    if ((self >> k) & 1u) continue;                       // solid source: nothing leaves it
                    if (bb || ((destf >> (k + cx + 1)) & 1u)) ownp[k] = g[i][k];   // bounced link
                    else {
                        int xd = c.x0 + k + cx;
                        xd = (xd < 0) ? p.nx - 1 : (xd >= p.nx ? 0 : xd);
                        rowp[xd] = g[i][k];
                    }
                }
                if constexpr (V > 1 && cx == 1) {
                    if (!bb && !c.edgeL && !(selff & 1u) && !((destf >> 1) & 1u)) rowp[c.x0] = nb;
                }
                if constexpr (V > 1 && cx == -1) {
                    if (!bb && !c.edgeR && !((selff >> (V + 1)) & 1u) && !((destf >> V) & 1u))
                        rowp[c.x0 + V - 1] = nb;
                }
            }
        });
    }
}

// ---------------------------------------------------------------------------------------------
// Hardware approximations (MUFU.RCP / MUFU.SQRT, <= 1 ulp).  Used only where the error enters at
// second order in the Mach number or multiplies the non-equilibrium part (DESIGN.md
// "Arithmetic form"): 1/rho in the quadratic terms, the two square roots and the reciprocal of
// the relaxation time.  Momentum is carried as j = rho u, so no result depends on
// rho * (1/rho) == 1.
// ---------------------------------------------------------------------------------------------
__device__ __forceinline__ float rcp_approx(float x)
{
    float r;
    asm("rcp.approx.ftz.f32 %0, %1;" : "=f"(r) : "f"(x));
    return r;
}
__device__ __forceinline__ float sqrt_approx(float x)
{
    float r;
    asm("sqrt.approx.ftz.f32 %0, %1;" : "=f"(r) : "f"(x));
    return r;
}

// ---------------------------------------------------------------------------------------------
// S2-S4: moments of the shifted populations, predictor velocity, forest drag, corrected
// velocity and total force of one cell (Eqs. 5-7, 13; Alg. 1).
// Pair sums/differences s_k = g_a + g_b, d_k = g_a - g_b over the 9 opposite pairs feed both the
// moments and the collision.
// ---------------------------------------------------------------------------------------------
struct Cell {
    float drho, rho, inv_rho;
    float jx, jy, jz;   // force-corrected momentum rho u = sum f c + F/2 (Eq. 6)
    float jxr;          // jx - J0: the same about the row's momentum reference
    float ux, uy, uz;   // force-corrected velocity (the sample S)
    float Fx, Fy, Fz;   // total force density F_b + F_f
    float Pxx, Pyy, Pzz, Pxy, Pyz, Pxz; // sum g_i c c  (= Pi - I/3)
};

// Momentum reference (arithmetic form only).  With omega close to 2
// the collision reflects the momentum channel, j* = (1 - w) m + w j, so a rounding error in the
// computed j - the 10-term sum at the magnitude of the mean flow, the product 3 w j, the inexact
// weights 1/18, 1/36 - returns doubled every step, and in a smooth flow with the same sign: a
// drift proportional to |u| (measured 1e-5 |u| after 100 steps).  The linear odd part of any
// reference equilibrium, ref_i = w_i 3 c_ix J0, passes through the collision unchanged
// ((1 - w) ref + w ref = ref), so the x-moving populations are taken about it: g'_i = g_i - ref_i
// before the moments, the collision acts on j' = j - J0 (small), and ref_i is added back in the
// final sum.  J0 is a per-row constant with few mantissa bits (r = J0/12 = ref of a diagonal
// population, 2r = ref of an axis population are exact); it changes rounding only, never the
// exact-arithmetic result.
template <int V>
__device__ __forceinline__ void mom_ref_shift(float (&g)[Q][V], int k, float r)
{
    const float r1 = 2.0f * r;
    g[1][k] -= r1; g[2][k] += r1;
    g[7][k] -= r; g[8][k] += r;
    g[9][k] -= r; g[10][k] += r;
    g[11][k] -= r; g[12][k] += r;
    g[13][k] -= r; g[14][k] += r;
}

// g: populations of the cell with mom_ref_shift(r) applied; r = J0 / 12 of the row.
template <int V>
__device__ __forceinline__ Cell moments(const KParams &p, const float (&g)[Q][V], int k, float cda, float r)
{
    Cell m;
    const float s1 = g[1][k] + g[2][k], d1 = g[1][k] - g[2][k];
    const float s3 = g[3][k] + g[4][k], d3 = g[3][k] - g[4][k];
    const float s5 = g[5][k] + g[6][k], d5 = g[5][k] - g[6][k];
    const float s7 = g[7][k] + g[8][k], d7 = g[7][k] - g[8][k];
    const float s9 = g[9][k] + g[10][k], d9 = g[9][k] - g[10][k];
    const float s11 = g[11][k] + g[12][k], d11 = g[11][k] - g[12][k];
    const float s13 = g[13][k] + g[14][k], d13 = g[13][k] - g[14][k];
    const float s15 = g[15][k] + g[16][k], d15 = g[15][k] - g[16][k];
    const float s17 = g[17][k] + g[18][k], d17 = g[17][k] - g[18][k];
    const float sxy = s7 + s9, sxz = s11 + s13, syz = s15 + s17;
    m.drho = g[0][k] + ((s1 + s3) + (s5 + sxy)) + (sxz + syz);          // Eq. 5 minus 1
    const float mx = (d1 + d7) + (d9 + d11) + d13;                      // Eq. 6 (bare momentum)
    const float my = (d3 + d7) + (d15 + d17) - d9;
    const float mz = (d5 + d11) + (d15 - d13) - d17;
    m.Pxx = s1 + sxy + sxz;                                              // Eq. 7 minus I/3
    m.Pyy = s3 + sxy + syz;
    m.Pzz = s5 + sxz + syz;
    m.Pxy = s7 - s9;
    m.Pxz = s11 - s13;
    m.Pyz = s15 - s17;
    m.rho = 1.0f + m.drho;
    m.inv_rho = rcp_approx(m.rho);
    // Alg. 1: local momentum with the driving force (Eq. 6; R7)
    m.jxr = mx + 0.5f * p.Fbx;
    m.jx = m.jxr + 12.0f * r;
    m.jy = my + 0.5f * p.Fby;
    m.jz = mz + 0.5f * p.Fbz;
    m.Fx = p.Fbx; m.Fy = p.Fby; m.Fz = p.Fbz;
    if (cda > 0.f) {
        // Alg. 1, Eq. 13: F_f = -C_D a_f(y) |u*| u*, no rho factor (R4), streamwise only (R5)
        const float usx = m.jx * m.inv_rho, usy = m.jy * m.inv_rho, usz = m.jz * m.inv_rho;
        const float coef = -cda * sqrt_approx(usx * usx + usy * usy + usz * usz);
        const float Ffx = coef * usx;
        // Alg. 1: correct the velocity with the forest force (explicit; R6)
        m.jx += 0.5f * Ffx; m.jxr += 0.5f * Ffx; m.Fx += Ffx;
        if (p.drag_vector) {
            const float Ffy = coef * usy, Ffz = coef * usz;
            m.jy += 0.5f * Ffy; m.Fy += Ffy;
            m.jz += 0.5f * Ffz; m.Fz += Ffz;
        }
    }
    m.ux = m.jx * m.inv_rho; m.uy = m.jy * m.inv_rho; m.uz = m.jz * m.inv_rho;
    return m;
}

// S5-S6: Smagorinsky tau_total (Eqs. 10-12; R8, R9) and the forced BGK collision (Eqs. 1-4; R1,
// R10) in even/odd pair form on the shifted populations, momentum form (j = rho u):
//   g*_i = (1-w) g_i + w (f_eq,i - w_i) + F_i,                     w = 1/tau_total
//   f_eq,i - w_i = w_i [ drho + 3 c.j + 4.5 (c.u)(c.j) - 1.5 u.j ],
//   F_i = (1 - w/2) w_i [ 3 c.F - 3 u.F + 9 (c.u)(c.F) ].
// Per pair (i, opp i):  even part  w_i [ e0 + (c.u)(c.h) ],  h = 4.5 w j + 9 (1-w/2) F
//                       odd part   w_i  c.k,                 k = 3 w j + 3 (1-w/2) F.
// The x-moving populations come in about the momentum reference (mom_ref_shift) and go out
// plain: their odd part is built from j' = jx - J0 and ref_i is added back in the same sum.
// Row-table SGS models (lbm_set_sgs_rows; "other SGS models"): with a per-row
// constant C_j and a per-row mean shear Sbar_j the closure nu_t = C_j (|S| - Sbar_j)_+ keeps the
// closed form of Eq. 12 with tau0 replaced by tau0 - 3 C_j Sbar_j, clipped below at tau0.
template <int V, bool SGS>
__device__ __forceinline__ void collide(const KParams &p, float (&g)[Q][V], int k, const Cell &m, float r, int y)
{
    const float ux = m.ux, uy = m.uy, uz = m.uz;
    const float third_drho = m.drho * (1.0f / 3.0f);
    const float nxx = m.Pxx - third_drho - m.jx * ux;   // Pi_neq = Pi - Pi_eq (L69)
    const float nyy = m.Pyy - third_drho - m.jy * uy;
    const float nzz = m.Pzz - third_drho - m.jz * uz;
    const float nxy = m.Pxy - m.jx * uy;
    const float nyz = m.Pyz - m.jy * uz;
    const float nxz = m.Pxz - m.jx * uz;
    const float QQ = (nxx * nxx + nyy * nyy + nzz * nzz) + 2.0f * (nxy * nxy + nyz * nyz + nxz * nxz);
    const float Qh = sqrt_approx(QQ);                                                      // Eq. 11
    float tau;
    if constexpr (SGS) {
        const float2 sg = __ldg(p.sgs + y);
        tau = fmaxf(0.5f * (sg.x + sqrt_approx(sg.x * sg.x + sg.y * Qh * m.inv_rho)), p.tau0);
    } else {
        tau = 0.5f * (p.tau0 + sqrt_approx(p.tau0sq + p.ksmag * Qh * m.inv_rho));          // Eq. 12
    }
    const float w = rcp_approx(tau);
    const float omw = 1.0f - w;
    const float gp = 1.0f - 0.5f * w;                                           // Guo prefactor (R10)
    const float uj = ux * m.jx + uy * m.jy + uz * m.jz;
    const float uF = ux * m.Fx + uy * m.Fy + uz * m.Fz;
    const float e0 = w * (m.drho - 1.5f * uj) - 3.0f * gp * uF;
    const float a2 = 4.5f * w, b2 = 9.0f * gp, a1 = 3.0f * w, b1 = 3.0f * gp;
    const float hx = a2 * m.jx + b2 * m.Fx, hy = a2 * m.jy + b2 * m.Fy, hz = a2 * m.jz + b2 * m.Fz;
    const float kx = a1 * m.jxr + b1 * m.Fx, ky = a1 * m.jy + b1 * m.Fy, kz = a1 * m.jz + b1 * m.Fz;
    constexpr float W0 = 1.0f / 3.0f, W1 = 1.0f / 18.0f, W2 = 1.0f / 36.0f;
    g[0][k] = omw * g[0][k] + W0 * e0;
    // axis pairs: c.u = u_a, c.h = h_a, c.k = k_a
    const float e1 = W1 * e0, e2 = W2 * e0;
#define LBM_PAIR(A, B, EV, OD)                      \
    {                                               \
        const float ev = (EV), od = (OD);           \
        g[A][k] = omw * g[A][k] + (ev + od);        \
        g[B][k] = omw * g[B][k] + (ev - od);        \
    }
    LBM_PAIR(1, 2, e1 + (W1 * ux) * hx, W1 * kx + 2.0f * r)
    LBM_PAIR(3, 4, e1 + (W1 * uy) * hy, W1 * ky)
    LBM_PAIR(5, 6, e1 + (W1 * uz) * hz, W1 * kz)
    const float vx = W2 * ux, vy = W2 * uy, vz = W2 * uz;   // weight folded into c.u
    const float qx = W2 * kx + r, qy = W2 * ky, qz = W2 * kz;   // weight folded into c.k (+ ref)
    LBM_PAIR(7, 8, e2 + (vx + vy) * (hx + hy), qx + qy)
    LBM_PAIR(9, 10, e2 + (vx - vy) * (hx - hy), qx - qy)
    LBM_PAIR(11, 12, e2 + (vx + vz) * (hx + hz), qx + qz)
    LBM_PAIR(13, 14, e2 + (vx - vz) * (hx - hz), qx - qz)
    LBM_PAIR(15, 16, e2 + (vy + vz) * (hy + hz), qy + qz)
    LBM_PAIR(17, 18, e2 + (vy - vz) * (hy - hz), qy - qz)
#undef LBM_PAIR
}

// ---------------------------------------------------------------------------------------------
// S8: stage 1 of the plane statistics - x-row sums of the sample S (L200, L251; R18).
// Columns: u, v, w, uu, vv, ww, uv, vw, uw, rho-1, all about the per-row centre `shift`.
// The block owns blockDim.y row segments; each is reduced with warp shuffles (+ shared memory
// across the warps of a segment) and stored, without atomics, to
//   partial[(y*NSTAT + k) * (nz*pchunks) + z*pchunks + chunk].
// ---------------------------------------------------------------------------------------------
__device__ __forceinline__ void stats_add(float (&s)[NSTAT], const Cell &m)
{
    s[0] += m.ux; s[1] += m.uy; s[2] += m.uz;
    s[3] += m.ux * m.ux; s[4] += m.uy * m.uy; s[5] += m.uz * m.uz;
    s[6] += m.ux * m.uy; s[7] += m.uy * m.uz; s[8] += m.ux * m.uz;
    s[9] += m.drho;
}

// Re-centre a thread's raw sums over n cells about (u0, v0, w0): sum (a-a0)(b-b0) =
// sum ab - a0 sum b - b0 sum a + n a0 b0.  Done once per thread, after the cell loop (the centre is
// not live across the loop), so that the cross-thread reduction works on small numbers.
__device__ __forceinline__ void stats_recentre(float (&s)[NSTAT], float n, float u0, float v0, float w0)
{
    const float a = s[0], b = s[1], c = s[2];
    s[3] += u0 * (n * u0 - 2.0f * a);
    s[4] += v0 * (n * v0 - 2.0f * b);
    s[5] += w0 * (n * w0 - 2.0f * c);
    s[6] += u0 * (n * v0 - b) - v0 * a;
    s[7] += v0 * (n * w0 - c) - w0 * b;
    s[8] += u0 * (n * w0 - c) - w0 * a;
    s[0] = a - n * u0; s[1] = b - n * v0; s[2] = c - n * w0;
}

// Sum each of the 10 columns over the 32 lanes of a warp: recursive-halving butterfly, 12
// shuffles (split 5|5, 3|3, 2|2, 1|1, then a plain exchange).  Afterwards the lanes 0, 2, 4, 8,
// 10 hold columns 0..4 and lanes 16, 18, 20, 24, 26 columns 5..9: `owner` lanes carry the total
// of column `col` in `v4`.
__device__ __forceinline__ void stats_warp_butterfly(const float (&s)[NSTAT], int lane, float &v4, bool &owner, int &col)
{
    const bool b16 = lane & 16, b8 = lane & 8, b4 = lane & 4, b2 = lane & 2;
    float v1[6], v2[4], v3[2];
#pragma unroll
    for (int k = 0; k < 5; ++k) {
        const float keep = b16 ? s[k + 5] : s[k], send = b16 ? s[k] : s[k + 5];
        v1[k] = keep + __shfl_xor_sync(0xffffffffu, send, 16);
    }
    v1[5] = 0.f;
#pragma unroll
    for (int k = 0; k < 3; ++k) {
        const float keep = b8 ? v1[k + 3] : v1[k], send = b8 ? v1[k] : v1[k + 3];
        v2[k] = keep + __shfl_xor_sync(0xffffffffu, send, 8);
    }
    v2[3] = 0.f;
#pragma unroll
    for (int k = 0; k < 2; ++k) {
        const float keep = b4 ? v2[k + 2] : v2[k], send = b4 ? v2[k] : v2[k + 2];
        v3[k] = keep + __shfl_xor_sync(0xffffffffu, send, 4);
    }
    v4 = (b2 ? v3[1] : v3[0]) + __shfl_xor_sync(0xffffffffu, b2 ? v3[0] : v3[1], 2);
    v4 += __shfl_xor_sync(0xffffffffu, v4, 1);
    const int q = (b8 ? 3 : 0) + (b4 ? 2 : 0) + (b2 ? 1 : 0);
    owner = !(lane & 1) && q < 5 && !(b8 && b4) && !(b4 && b2);
    col = (b16 ? 5 : 0) + q;
}

__device__ __forceinline__ void stats_row_reduce(const KParams &p, const Ctx &c, float (&s)[NSTAT])
{
    __shared__ float sred[MAX_THREADS / 32][NSTAT];
    __shared__ float srow[MAX_THREADS][NSTAT + 1];
    const int TX = blockDim.x, tx = threadIdx.x, ty = threadIdx.y;
    const int lin = ty * TX + tx, warp = lin >> 5, lane = lin & 31;
    const long long pstride = (long long)p.nz * p.pchunks;
    float *out = p.partial + ((long long)c.y * NSTAT) * pstride + (long long)c.z * p.pchunks + c.chunk;
    if ((TX & 31) == 0) {
        // every warp lies inside one row segment
        float v4;
        bool owner;
        int col;
        stats_warp_butterfly(s, lane, v4, owner, col);
        const int wpr = TX >> 5;
        if (wpr == 1) {
            if (owner) out[(long long)col * pstride] = v4;
        } else if (p.wpart) {
            if (owner) out[(long long)col * pstride + (long long)c.chunk * (wpr - 1) + (tx >> 5)] = v4;
        } else {
            if (owner) sred[warp][col] = v4;
            __syncthreads();
            if (tx < NSTAT) {
                float v = 0.f;
                for (int w2 = 0; w2 < wpr; ++w2) v += sred[ty * wpr + w2][tx];
                out[(long long)tx * pstride] = v;
            }
        }
    } else if (TX < 32 && (TX & (TX - 1)) == 0) {
        // several whole row segments per warp: butterfly inside aligned groups of TX lanes
#pragma unroll
        for (int k = 0; k < NSTAT; ++k) {
            for (int o = TX >> 1; o > 0; o >>= 1) s[k] += __shfl_xor_sync(0xffffffffu, s[k], o);
        }
        if (tx == 0) {
#pragma unroll
            for (int k = 0; k < NSTAT; ++k) out[(long long)k * pstride] = s[k];
        }
    } else {
        // irregular width (the paper's 350- and 372-cell meshes: 175, 93 threads per row): through
        // shared memory; every FULL warp of the block then reduces whole row segments - each lane sums
        // the entries lane, lane + 32, ... of the ten columns, the butterfly finishes - and the
        // owner lanes store.  Blocks smaller than a warp sum serially.
        const int TY = blockDim.y;
#pragma unroll
        for (int k = 0; k < NSTAT; ++k) srow[lin][k] = s[k];
        __syncthreads();
        const int nfull = (TX * TY) >> 5;
        if (nfull == 0) {
            for (int k = tx; k < NSTAT; k += TX) {   // TX may be smaller than NSTAT
                float v = 0.f;
                for (int q = 0; q < TX; ++q) v += srow[ty * TX + q][k];
                out[(long long)k * pstride] = v;
            }
        } else if (warp < nfull) {
            const int row0 = c.z * p.ny + c.y - ty;          // row of segment 0 of this block
            for (int seg = warp; seg < TY; seg += nfull) {
                float v[NSTAT];
#pragma unroll
                for (int k = 0; k < NSTAT; ++k) v[k] = 0.f;
                for (int q = lane; q < TX; q += 32) {
#pragma unroll
                    for (int k = 0; k < NSTAT; ++k) v[k] += srow[seg * TX + q][k];
                }
                float v4;
                bool owner;
                int col;
                stats_warp_butterfly(v, lane, v4, owner, col);
                const int row = row0 + seg, z = row / p.ny, y = row - z * p.ny;
                if (owner)
                    p.partial[((long long)y * NSTAT + col) * pstride + (long long)z * p.pchunks + c.chunk] = v4;
            }
        }
    }
}

// ---------------------------------------------------------------------------------------------
// The step kernel.  grid = (row blocks, x chunks), block = (TX, TY) <= 256 threads.
// ---------------------------------------------------------------------------------------------
template <int V> struct Occ { static constexpr int minb = (V == 4) ? 2 : (V == 2 ? 3 : 4); };
// (A larger register budget for the geometry variants - 168 registers, three blocks of 128
// threads per SM - was measured and is slower than 128 registers with four blocks: 0.58 vs 0.47 ms
// on cfg3 with statistics; profiles/r02_README.md.)
constexpr int MASK_THREADS = 256;
template <int V, bool MASK> struct Bounds {
    static constexpr int threads = MAX_THREADS;
    static constexpr int minb = Occ<V>::minb;
};

// S2-S6 (+ the S8 sample) of the thread's V cells in registers: g holds the streamed populations on
// entry and the post-collision ones on exit, s the thread's ten statistics sums.  Shared by the
// per-thread and the TMA step kernels (bit-identical by construction).
template <int V, bool STATS, bool MASK, bool SGS>
__device__ __forceinline__ void cells_update(const KParams &p, float (&g)[Q][V], float (&s)[NSTAT], float cda,
                                             unsigned fidx, float jr, unsigned long long S, int y)
{
    // (The same arithmetic on PAIRS of cells with Blackwell's packed fp32 instructions - FADD2 / FMUL2 /
    // FFMA2, `__ffma2_rn` and friends: 105 instead of 243 fp32 instructions per cell - was built and
    // measured in round 2: parity unchanged, but the pairs need 19 more live registers than the
    // kernel has (40-140 B of spills with the statistics fused) and the kernel waits for DRAM, not
    // for the fp32 pipe: cfg5 38.2 against 41.6 GLUPS with statistics, 41.4 against 42.5 without.  Dropped.)
    if constexpr (STATS) {
#pragma unroll
        for (int k = 0; k < NSTAT; ++k) s[k] = 0.f;
    }
#pragma unroll
    for (int k = 0; k < V; ++k) {
        mom_ref_shift<V>(g, k, jr);
        const Cell m = moments<V>(p, g, k, cell_cda<MASK>(p, cda, fidx, k), jr);
        if constexpr (STATS) {
            // solid cells are left out of the plane sums (the divisor stays nx*nz, as in the
            // oracle's O10); with a mask the host never sets an accumulation centre (p.shift)
            if (!MASK || !((solid_self<V>(S) >> k) & 1u)) stats_add(s, m);
        }
        collide<V, SGS>(p, g, k, m, jr, y);
    }
}

template <int V, int RM, int WM, bool STATS, bool MASK, bool SGS>
__device__ __forceinline__ void step_body(const KParams &p)
{
    const Ctx c = make_ctx<V>(p, p.z0 * p.ny);
    // Geometry body (only blocks flagged by blockflag_kernel come here): the nine-row gather of the
    // solid bits is requested BEFORE the 19 population loads, so both travel together and the only
    // dependent round trip left is the own-cell loads of the links that bounce.  A warp none of
    // whose lanes has a solid cell within one step runs the unmasked load/store code; the decision
    // is warp-uniform, so the full-mask shuffles inside load_dir/store_dir stay converged.
    unsigned long long S = 0ull;
    if constexpr (MASK) S = solid_gather_rows<V>(p, c);
    float g[Q][V];
    load_all<V, RM>(p, c, g);
    bool geom = false;
    if constexpr (MASK) {
        geom = __any_sync(0xffffffffu, S != 0ull);
        if (geom) solid_fix_loads<V, RM>(p, c, g, S);
    }
    const float cda = __ldg(p.cda + c.y);
    const unsigned fidx = forest_idx<V, MASK>(p, c);
    const float jr = __ldg(p.jref + c.y);
    float s[NSTAT];
    cells_update<V, STATS, MASK, SGS>(p, g, s, cda, fidx, jr, S, c.y);
    const Ctx c2 = (WM == WR_PUSH || WM == WR_XO) ? make_ctx<V>(p, p.z0 * p.ny, true) : c;
    // the accumulation centre of the row is prefetched into L1 before the stores are issued and
    // loaded after them: loaded where it is used its latency was 5-7 % of the warp time (ncu source
    // page, round 2; the streaming loads keep evicting the small table from L1), and holding it in
    // registers across the store phase spills in the x-balanced even step
    if constexpr (STATS) {
        if (p.shift) asm volatile("prefetch.global.L1 [%0];" ::"l"(reinterpret_cast<const float4 *>(p.shift) + c2.y));
    }
    if (MASK && geom) store_all<V, WM, MASK>(p, c2, g, S);
    else store_all<V, WM, false>(p, c2, g);
    if constexpr (STATS) {
        if (p.shift) {
            const float4 sh = __ldg(reinterpret_cast<const float4 *>(p.shift) + c2.y);
            stats_recentre(s, (float)V, sh.x, sh.y, sh.z);
        }
        stats_row_reduce(p, c2, s);
    }
}

// Geometry handles: a thread block none of whose cells has a solid cell within one step, nor a coded
// forest cell, runs the plain body - the same code as the kernel without MASK (the per-block flag
// is built by blockflag_kernel whenever the geometry or the block shape changes).  The flag is one
// byte per block, read before anything else; in sparse geometry almost every block takes the plain
// path, so the instruction cache sees one body.
template <int V, int RM, int WM, bool STATS, bool MASK = false, bool SGS = false>
__global__ void __launch_bounds__(Bounds<V, MASK>::threads, Bounds<V, MASK>::minb) step_kernel(const KParams p)
{
    pdl_enter();
    // (The geometry body as a __noinline__ function of its own, so that the plain body keeps the
    // register allocation of the kernel without MASK, was measured: slower - cfg3 boxes + statistics
    // 39.2 against 39.7 GLUPS, cfg4 all-fluid mask -4.7 % against -0.7 % - and dropped.)
    if constexpr (MASK) {
        if (__ldg(p.bflag + block_linear(p)) == 0) {
            step_body<V, RM, WM, STATS, false, SGS>(p);
            return;
        }
    }
    step_body<V, RM, WM, STATS, MASK, SGS>(p);
}

// One thread per thread block of the step launch (block = tx_cells x ty rows, nchunk blocks per
// row): flag = any bit of the dilated solid mask, or any coded forest cell, inside the block.
static __global__ void blockflag_kernel(const KParams p, int tx_cells, int ty, unsigned char *out, long long nblocks)
{
    const long long b = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (b >= nblocks) return;
    const long long rb = b / p.nchunk;
    const int chunk = (int)(b - rb * p.nchunk);
    const int x0 = chunk * tx_cells, x1 = x0 + tx_cells;
    unsigned any = 0u;
    for (int r = 0; r < ty; ++r) {
        const long long row = rb * ty + r;
        const unsigned *m = p.solid_nb + row * p.nxw;
        for (int w = x0 >> 5; w <= (x1 - 1) >> 5; ++w) {
            unsigned v = m[w];
            const int lo = w << 5;
            if (lo < x0) v &= ~0u << (x0 - lo);
            if (lo + 32 > x1) v &= ~0u >> (lo + 32 - x1);
            any |= v;
        }
        if (p.fidx && p.frow[row % p.ny])
            for (int x = x0; x < x1; ++x) any |= p.fidx[row * p.nx + x];
    }
    out[b] = any ? 1 : 0;
}

// Sample S_k without changing the state (R19): the front half of the step (S1-S4).  Writes
// rho/u when the pointers are given and the stage-1 sums when p.partial is given.
// Covers rows [z0*ny, z1*ny).
template <int V, int RM, bool MASK = false>
__global__ void __launch_bounds__(Bounds<V, MASK>::threads, Bounds<V, MASK>::minb) macros_kernel(const KParams p)
{
    const Ctx c = make_ctx<V>(p, p.z0 * p.ny);
    float g[Q][V];
    load_all<V, RM>(p, c, g);
    unsigned long long S = 0ull;
    if constexpr (MASK) {
        S = solid_gather<V>(p, c, solid_nb_word(p, c));
        if (__any_sync(0xffffffffu, S != 0ull)) solid_fix_loads<V, RM>(p, c, g, S);
    }
    const float cda = __ldg(p.cda + c.y);
    const unsigned fidx = forest_idx<V, MASK>(p, c);
    float s[NSTAT];
#pragma unroll
    for (int k = 0; k < NSTAT; ++k) s[k] = 0.f;
    float r[V], ux[V], uy[V], uz[V];
#pragma unroll
    for (int k = 0; k < V; ++k) {
        const Cell m = moments<V>(p, g, k, cell_cda<MASK>(p, cda, fidx, k), 0.f);
        const bool solid = MASK && ((solid_self<V>(S) >> k) & 1u);
        if (!solid) stats_add(s, m);
        r[k] = solid ? 1.0f : m.rho;             // solid cells report the rest state
        ux[k] = solid ? 0.f : m.ux; uy[k] = solid ? 0.f : m.uy; uz[k] = solid ? 0.f : m.uz;
        if (!isfinite(r[k]) && p.diverged && c.z >= p.zv0 && c.z < p.zv1) *p.diverged = 1;   // LBM_EDIVERGED sentinel
    }
    const long long off = (long long)(c.y + p.ny * (c.z - p.z0)) * p.nx + c.x0 + p.zoff;
    if (p.rho_out) stv<V>(p.rho_out + off, r);
    if (p.u_out) {
        stv<V>(p.u_out + off, ux);
        stv<V>(p.u_out + p.Nio + off, uy);
        stv<V>(p.u_out + 2 * p.Nio + off, uz);
    }
    if (p.partial) {
        if (p.shift) {
            const float4 sh = __ldg(reinterpret_cast<const float4 *>(p.shift) + c.y);
            stats_recentre(s, (float)V, sh.x, sh.y, sh.z);
        }
        stats_row_reduce(p, c, s);
    }
}

// splitmix64 output function of seed + (ctr+1)*golden.
__host__ __device__ __forceinline__ unsigned long long mix64(unsigned long long seed, unsigned long long ctr)
{
    unsigned long long z = seed + (ctr + 1ULL) * 0x9E3779B97F4A7C15ULL;
    z = (z ^ (z >> 30)) * 0xBF58476D1CE4E5B9ULL;
    z = (z ^ (z >> 27)) * 0x94D049BB133111EBULL;
    return z ^ (z >> 31);
}

// State 0 (R17): g_i = f_eq,i(rho, u) - w_i with (rho, u) from the caller's fields or from the
// synthetic recipe (R16), written in the representation the storage scheme wants
// (WR_LOCAL: two-lattice; WR_PUSH: AA at even t).  Covers rows [z0*ny, z1*ny).
template <int V, int WM, bool MASK = false>
__global__ void __launch_bounds__(MAX_THREADS, Occ<V>::minb) init_kernel(const KParams p)
{
    const Ctx c = make_ctx<V>(p, p.z0 * p.ny);
    unsigned long long S = 0ull;
    if constexpr (MASK) S = solid_gather<V>(p, c, solid_nb_word(p, c));
    float g[Q][V];
    const long long cell0 = (long long)(c.y + p.ny * c.z) * p.nx + c.x0;
    const long long off = (long long)(c.y + p.ny * (c.z - p.z0)) * p.nx + c.x0 + p.zoff;
#pragma unroll
    for (int k = 0; k < V; ++k) {
        float rho, ux, uy, uz;
        if (p.rho_in) {
            rho = p.rho_in[off + k];
            ux = p.u_in[off + k]; uy = p.u_in[p.Nio + off + k]; uz = p.u_in[2 * p.Nio + off + k];
        } else {
            // global cell index of the recipe (a z slab initialises its part of the global field)
            int zg = (c.z + p.zg0) % p.nzg;
            if (zg < 0) zg += p.nzg;
            const unsigned long long cell = (unsigned long long)((long long)(c.y + p.ny * zg) * p.nx + c.x0 + k);
            const double inv53 = 1.0 / 9007199254740992.0;
            const double r0 = (double)(mix64(p.seed, 3ULL * cell + 0ULL) >> 11) * inv53;
            const double r1 = (double)(mix64(p.seed, 3ULL * cell + 1ULL) >> 11) * inv53;
            const double r2 = (double)(mix64(p.seed, 3ULL * cell + 2ULL) >> 11) * inv53;
            rho = 1.0f;
            ux = (float)((double)p.uprof[c.y] + p.noise_amp * (2.0 * r0 - 1.0));
            uy = (float)(p.noise_amp * (2.0 * r1 - 1.0));
            uz = (float)(p.noise_amp * (2.0 * r2 - 1.0));
        }
        if (MASK && ((solid_self<V>(S) >> k) & 1u)) { rho = 1.0f; ux = uy = uz = 0.f; }  // rest state
        const float drho = rho - 1.0f;
        const float uu = ux * ux + uy * uy + uz * uz;
        const float e0 = drho - 1.5f * rho * uu;
        g[0][k] = (1.0f / 3.0f) * e0;
        static_for<1, Q>([&](auto ic) {
            constexpr int i = decltype(ic)::value;
            constexpr float wgt = (i < 7) ? (1.0f / 18.0f) : (1.0f / 36.0f);
            constexpr float ex = (float)Lat::cx[i], ey = (float)Lat::cy[i], ez = (float)Lat::cz[i];
            const float cu = ex * ux + ey * uy + ez * uz;
            g[i][k] = wgt * (e0 + rho * cu * (3.0f + 4.5f * cu));
        });
    }
    store_all<V, WM, MASK>(p, c, g, S);
}

// Plain "state k" populations [19][N] (the layout lbm_get_state writes) into whatever
// representation the storage scheme / time parity wants: WR_LOCAL (two-lattice), WR_LOCAL_OPP
// (AA, t odd), WR_PUSH (AA, t even).  Solid cells are written as the rest state.
template <int V, int WM, bool MASK = false>
__global__ void __launch_bounds__(MAX_THREADS, Occ<V>::minb) setstate_kernel(const KParams p, const float *in)
{
    const Ctx c = make_ctx<V>(p, p.z0 * p.ny);
    unsigned long long S = 0ull;
    if constexpr (MASK) S = solid_gather<V>(p, c, solid_nb_word(p, c));
    float g[Q][V];
    const long long cell0 = (long long)(c.y + p.ny * c.z) * p.nx + c.x0;
    static_for<0, Q>([&](auto ic) {
        constexpr int i = decltype(ic)::value;
        ldv<V>(in + (long long)i * p.N + cell0, g[i]);
    });
    store_all<V, WM, MASK>(p, c, g, S);
}

__device__ __forceinline__ bool solid_at(const KParams &p, int x, int y, int z)
{
    if (!p.solid) return false;
    return (p.solid[(long long)(y + p.ny * z) * p.nxw + (x >> 5)] >> (x & 31)) & 1u;
}

// Where the AA "push" representation (t even) keeps population i of cell (x, y, z): slot and cell of
// store_all<WR_PUSH> - the neighbour, or the own cell's opposite slot when the link bounces off a
// wall face or a solid cell, or the mirrored slot of the tangential neighbour at a free-slip face.
struct PushLoc { int slot; long long cell; bool self; };
template <int i>
__device__ __forceinline__ PushLoc push_target(const KParams &p, const unsigned *mask, int x, int y, int z)
{
    constexpr int cx = Lat::cx[i], cy = Lat::cy[i], cz = Lat::cz[i];
    const long long own = (long long)(y + p.ny * z) * p.nx + x;
    int slot = i, xd = x + cx, yd = y + cy, zd = z + cz;
    xd = (xd < 0) ? p.nx - 1 : (xd >= p.nx ? 0 : xd);
    zd = (zd < 0) ? p.nz - 1 : (zd >= p.nz ? 0 : zd);
    if (yd < 0) {
        if (p.bot == BC_BOT_PERIODIC) yd = p.ny - 1;
        else return {Lat::opp[i], own, true};
    } else if (yd >= p.ny) {
        if (p.top == BC_TOP_PERIODIC) yd = 0;
        else if (p.top == BC_TOP_SLIP) { slot = Lat::mir[i]; yd = y; }
        else return {Lat::opp[i], own, true};
    }
    if (mask && ((mask[(long long)(yd + p.ny * zd) * p.nxw + (xd >> 5)] >> (xd & 31)) & 1u)) return {Lat::opp[i], own, true};
    return {slot, (long long)(yd + p.ny * zd) * p.nx + xd, false};
}
__device__ __forceinline__ bool mask_bit(const unsigned *mask, const KParams &p, long long cell)
{
    const long long row = cell / p.nx;
    const int x = (int)(cell - row * p.nx);
    return (mask[row * p.nxw + (x >> 5)] >> (x & 31)) & 1u;
}

// Run-time change of the solid mask that keeps the flow ("Once the turbulence is
// developed, the boxes are removed ... The flow remains in the turbulent status afterwards").
// One thread per cell; only cells whose bit changes act.  `arr` is the array holding state t.
//   PUSH = false (two-lattice; AA at odd t): the representation does not depend on the mask; a cell
//          that turns solid is cleared to the rest state, a cell that turns fluid holds it already.
//   PUSH = true  (AA at even t): populations sit where the OLD mask sent them.  Between a changed
//          cell d and a neighbour n that is fluid before and after:
//            d turns fluid: n's population that had bounced off d (own slot of n) moves into d,
//                           and n's slot receives d's rest population (0);
//            d turns solid: n's population that had entered d bounces instead (moves to the own
//                           slot of n, replacing what d had pushed there); d is cleared.
//   AAX (x-balanced AA, either parity): the same, with every slot whose c_x is +1 kept one cell to the
//          left of the cell it belongs to (slot s of cell n sits at n - [c_sx = +1] e_x).
__device__ __forceinline__ long long left_of(const KParams &p, long long cell, bool shift)
{
    if (!shift) return cell;
    return (cell % p.nx == 0) ? cell + p.nx - 1 : cell - 1;
}
template <bool PUSH, bool AAX = false>
__global__ void mask_change_kernel(const KParams p, float *arr, const unsigned *oldm, const unsigned *newm)
{
    const long long d = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (d >= p.N) return;
    const bool was = mask_bit(oldm, p, d), is = mask_bit(newm, p, d);
    if (was == is) return;
    const int x = (int)(d % p.nx);
    const long long row = d / p.nx;
    const int y = (int)(row % p.ny), z = (int)(row / p.ny);
    if constexpr (PUSH) {
        static_for<1, Q>([&](auto ic) {
            constexpr int i = decltype(ic)::value;
            // the link d --i--> n under the geometry in which d is fluid
            const PushLoc t = push_target<i>(p, is ? oldm : newm, x, y, z);
            if (t.self) return;
            if (mask_bit(oldm, p, t.cell) || mask_bit(newm, p, t.cell)) return;   // n must be fluid before and after
            // n's own slot on this link (slot i, or its y mirror at a free-slip face: the same c_x)
            constexpr bool sh_n = AAX && Lat::cx[i] == 1, sh_d = AAX && Lat::cx[i] == -1;
            float *at_n = arr + (long long)t.slot * p.N + left_of(p, t.cell, sh_n);
            // where n's population enters d (slot opp(i))
            float *at_d = arr + (long long)Lat::opp[i] * p.N + left_of(p, d, sh_d);
            if (!is) { *at_d = *at_n; *at_n = 0.f; }                        // d turns fluid
            else *at_n = *at_d;                                             // d turns solid
        });
    }
    if (is) {
        static_for<0, Q>([&](auto ic) {
            constexpr int i = decltype(ic)::value;
            constexpr bool sh = AAX && Lat::cx[i] == 1;
            arr[(long long)i * p.N + left_of(p, d, sh)] = 0.f;
        });
    }
}

// Plain "state k" (post-collision, un-streamed) populations out of whatever representation the
// storage holds: out[i][cell] = g*_i(cell).  One cell per thread (checkpoint / tests only).
//   two-lattice          : src[i][x]
//   AA, t odd            : src[opp i][x]
//   AA, t even (PUSH)    : src[i][x + c_i] with the wall / free-slip / solid redirections of
//                          store_all; solid cells report the rest state (0)
//   AAX, t odd  (MODE 3) : src[opp i][x - 1 if c_x = -1 else x]
//   AAX, t even (MODE 4) : as PUSH in slot, y and z; in x: x - 1 if c_x = -1 else x
template <int MODE>
__global__ void state_kernel(const KParams p, float *out)
{
    const long long cell = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (cell >= p.N) return;
    const int x = (int)(cell % p.nx);
    const long long row = cell / p.nx;
    const int y = (int)(row % p.ny), z = (int)(row / p.ny);
    const bool self_solid = solid_at(p, x, y, z);
    static_for<0, Q>([&](auto ic) {
        constexpr int i = decltype(ic)::value;
        constexpr int cx = Lat::cx[i], cy = Lat::cy[i], cz = Lat::cz[i];
        constexpr int S_OPP = Lat::opp[i], S_MIR = Lat::mir[i];
        float v;
        // x-balanced AA: in every representation only the c_x = -1 populations sit one cell to the left
        constexpr int xdx = (cx == -1) ? -1 : 0;
        if constexpr (MODE == 0) v = p.src[(long long)i * p.N + cell];
        else if constexpr (MODE == 1) v = p.src[(long long)S_OPP * p.N + cell];
        else if constexpr (MODE == 3) {
            int xd = x + xdx;
            xd = (xd < 0) ? p.nx - 1 : xd;
            v = p.src[(long long)S_OPP * p.N + (cell - x + xd)];
        } else {
            int slot = i, xd = x + (MODE == 4 ? xdx : cx), yd = y + cy, zd = z + cz;
            int xt = x + cx;                                   // the cell the link leads to
            xt = (xt < 0) ? p.nx - 1 : (xt >= p.nx ? 0 : xt);
            xd = (xd < 0) ? p.nx - 1 : (xd >= p.nx ? 0 : xd);
            zd = (zd < 0) ? p.nz - 1 : (zd >= p.nz ? 0 : zd);
            if (yd < 0) {
                if (p.bot == BC_BOT_PERIODIC) yd = p.ny - 1;
                else { slot = S_OPP; xd = (MODE == 4) ? xd : x; yd = y; zd = z; }
            } else if (yd >= p.ny) {
                if (p.top == BC_TOP_PERIODIC) yd = 0;
                else if (p.top == BC_TOP_SLIP) { slot = S_MIR; yd = y; }
                else { slot = S_OPP; xd = (MODE == 4) ? xd : x; yd = y; zd = z; }
            }
            if (MODE == 2 && solid_at(p, xd, yd, zd)) { slot = S_OPP; xd = x; yd = y; zd = z; }
            // x-balanced: a link that bounces off a solid changes slot and row, not the x displacement
            if (MODE == 4 && solid_at(p, xt, yd, zd)) { slot = S_OPP; yd = y; zd = z; }
            v = p.src[(long long)slot * p.N + ((long long)(yd + p.ny * zd) * p.nx + xd)];
        }
        out[(long long)i * p.N + cell] = self_solid ? 0.f : v;
    });
}

// ---------------------------------------------------------------------------------------------
// S9: stage 2 of the statistics - reduce the row partials of one (y, k) over z (and x chunks)
// in fp64 with warp shuffles + shared memory and add into the running sums acc[y][k].
// grid = (ny, NSTAT), block = 256.  mode 0: accumulate; mode 1: prime the accumulation centre
// shift[y][0..2] with the current plane means instead.
// ---------------------------------------------------------------------------------------------
static __global__ void __launch_bounds__(256) stats_stage2_kernel(const float *__restrict__ partial, long long len,
                                                           double *acc, float *shift, int mode,
                                                           double inv_count, int *diverged)
{
    __shared__ double sm[8];
    pdl_enter();
    const int y = blockIdx.x, k = blockIdx.y;
    const float *src = partial + ((long long)y * NSTAT + k) * len;
    double t = 0.0;
    for (long long q = threadIdx.x; q < len; q += blockDim.x) t += (double)src[q];
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) t += __shfl_xor_sync(0xffffffffu, t, o);
    if ((threadIdx.x & 31) == 0) sm[threadIdx.x >> 5] = t;
    __syncthreads();
    if (threadIdx.x == 0) {
        double tot = 0.0;
        for (int w = 0; w < (int)(blockDim.x >> 5); ++w) tot += sm[w];
        if (mode == 0) {
            acc[y * NSTAT + k] += tot;
            if (k == NSTAT - 1 && !isfinite(tot)) *diverged = 1;
        } else if (k < 3) {
            const double mean = tot * inv_count;
            shift[y * 4 + k] = isfinite(mean) ? (float)mean : 0.f;
        }
    }
}

// ---------------------------------------------------------------------------------------------
// z-slab halo exchange: the five populations that cross a z face, of one x-y
// plane, to / from a contiguous buffer [5][ny][nx].  side 1: slots with c_z = +1 (i = 5, 11, 14, 15,
// 18), side 0: slots with c_z = -1 (i = 6, 12, 13, 16, 17).  pack reads plane `z`, unpack writes
// plane `z`.  Which plane and which slot set a face exchange moves depends on the storage scheme
// and the time parity (lbm_api.cu: halo_map).
//
// FILTER (unpack only): the single-array storages at even t keep population i of cell x at slot i
// of cell x + c_i ("push" representation), so what crosses the face is the neighbour rank's ghost
// plane, going into the slots of REAL cells of the boundary plane.  Only entries that a cell of the
// ghost plane has written may land: an entry whose source cell lies beyond a wall / lid face or is
// solid holds the destination cell's own bounced population and stays; nothing lands in a solid cell.
// ---------------------------------------------------------------------------------------------
// One launch serves one face (gridDim.y = 1) or both (gridDim.y = 2: blockIdx.y = 1 takes the
// second (z, side, buf) triple).
struct HaloFace { int z, side; float *buf; };
template <bool PACK, bool FILTER>
__global__ void halo_kernel(const KParams p, float *pops, HaloFace f0, HaloFace f1)
{
    pdl_enter();
    const HaloFace f = blockIdx.y ? f1 : f0;
    const int z = f.z, side = f.side;
    float *buf = f.buf;
    const long long plane = (long long)p.nx * p.ny;
    const long long q = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (q >= 5 * plane) return;
    const int j = (int)(q / plane);
    const long long r = q - (long long)j * plane;
    const int up[5] = {5, 11, 14, 15, 18}, dn[5] = {6, 12, 13, 16, 17};
    const int i = side ? up[j] : dn[j];
    if constexpr (FILTER) {
        const int cxs[Q] = {0, 1, -1, 0, 0, 0, 0, 1, -1, 1, -1, 1, -1, 1, -1, 0, 0, 0, 0};
        const int cys[Q] = {0, 0, 0, 1, -1, 0, 0, 1, -1, -1, 1, 0, 0, 0, 0, 1, -1, 1, -1};
        const int y = (int)(r / p.nx), x = (int)(r - (long long)y * p.nx);
        int ys = y - cys[i];
        if (ys < 0) {
            if (p.bot == BC_BOT_PERIODIC) ys = p.ny - 1; else return;       // the cell's own bounce off the wall
        } else if (ys >= p.ny) {
            if (p.top == BC_TOP_PERIODIC) ys = 0;
            else if (p.top == BC_TOP_SLIP) ys = y;                          // mirrored link from the same row
            else return;
        }
        // x-balanced AA: the entry at memory column x belongs to cell x + 1 when c_x = +1
        int xc = x + ((p.aax && cxs[i] == 1) ? 1 : 0);
        xc = (xc >= p.nx) ? 0 : xc;
        int xs = xc - cxs[i];
        xs = (xs < 0) ? p.nx - 1 : (xs >= p.nx ? 0 : xs);
        const int zs = side ? z - 1 : z + 1;                                 // the ghost plane it came from
        if (p.solid && (solid_at(p, xc, y, z) || solid_at(p, xs, ys, zs))) return;
    }
    float *cell = pops + (long long)i * p.N + (long long)z * plane + r;
    if (PACK) buf[q] = *cell; else *cell = buf[q];
}

} // namespace lbm
