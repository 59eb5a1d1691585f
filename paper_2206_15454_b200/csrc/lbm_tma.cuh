// lbm_tma.cuh — the fused step with the stream-in done by the Tensor Memory Accelerator.
//
// Same time step as lbm::step_kernel (Algorithm 1; the per-cell arithmetic, the
// stores and the statistics are the same code), different stream-in.  In step_kernel every thread
// fetches its own 4 cells with 128-bit loads and pays for the +-1 x shift of 10 of the 19
// directions (Eq. 1) with a 64-bit address computation, a shuffle, per-lane selects and a
// scalar edge load per direction.  Here a CTA owns a tile of 256 x R cells (R consecutive y rows
// of one z plane) and
//   1. one lane of every warp issues `cp.async.bulk.tensor` loads of the tile's R row segments of
//      its share of the 19 populations, from wherever the streaming step says they come from: the
//      box coordinate (x0, y - c_y, z - c_z, slot) carries the row and slot of the link (neighbour
//      row, bounce-back / free-slip slot, periodic wrap), all 19 x R boxes complete on one mbarrier;
//   2. the x shift is taken when the tile is read back: a thread's vector of direction i is its own
//      aligned LDS.128 with the element of the neighbouring thread (one LDS.32) shifted in; the one
//      element beyond the tile edge (with the periodic x wrap) is fetched by a scalar load into a
//      halo word.  (The TMA unit itself cannot take the shift: a box must start on a 16-byte
//      boundary of global memory - x0 - 1 raises an illegal-instruction fault, measured.)
//   3. moments / drag / Smagorinsky / collision, stores and fused statistics as in step_kernel.
// Several CTAs per SM overlap the phases.
//
// Requirements: 4 cells per thread layout (nx % 256 == 0), R | ny, no solid mask.
#pragma once
#include <cuda.h>

#include "lbm_launch.cuh"

namespace lbm {

constexpr int TMA_TX = TMA_BOX / 4;       // threads along x

static __constant__ signed char TMA_CX[Q] = {0, 1, -1, 0, 0, 0, 0, 1, -1, 1, -1, 1, -1, 1, -1, 0, 0, 0, 0};
static __constant__ signed char TMA_CY[Q] = {0, 0, 0, 1, -1, 0, 0, 1, -1, -1, 1, 0, 0, 0, 0, 1, -1, 1, -1};
static __constant__ signed char TMA_CZ[Q] = {0, 0, 0, 0, 0, 1, -1, 0, 0, 0, 0, 1, -1, -1, 1, 1, -1, -1, 1};
static __constant__ signed char TMA_OPP[Q] = {0, 2, 1, 4, 3, 6, 5, 8, 7, 10, 9, 12, 11, 14, 13, 16, 15, 18, 17};
static __constant__ signed char TMA_MIR[Q] = {0, 1, 2, 4, 3, 5, 6, 9, 10, 7, 8, 11, 12, 13, 14, 18, 17, 16, 15};

__device__ __forceinline__ uint32_t smem_addr(const void *p)
{
    return (uint32_t)__cvta_generic_to_shared(p);
}
__device__ __forceinline__ void mbar_init(uint64_t *bar, uint32_t count)
{
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_addr(bar)), "r"(count) : "memory");
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
}
__device__ __forceinline__ void mbar_arrive_expect_tx(uint64_t *bar, uint32_t bytes)
{
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_addr(bar)), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_wait(uint64_t *bar, uint32_t parity)
{
    uint32_t done;
    do {
        asm volatile(
            "{\n"
            ".reg .pred p;\n"
            "mbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n"
            "selp.u32 %0, 1, 0, p;\n"
            "}\n"
            : "=r"(done)
            : "r"(smem_addr(bar)), "r"(parity)
            : "memory");
    } while (!done);
}
// global (tensor map, box at {x, y, z, slot}) -> shared, completes `bytes` on the mbarrier
__device__ __forceinline__ void tma_load_box(void *dst, const CUtensorMap *map, int x, int y, int z, int slot,
                                             uint64_t *bar)
{
    asm volatile(
        "cp.async.bulk.tensor.4d.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1, {%3, %4, %5, %6}], [%2];"
        ::"r"(smem_addr(dst)), "l"(reinterpret_cast<uint64_t>(map)), "r"(smem_addr(bar)), "r"(x), "r"(y), "r"(z), "r"(slot)
        : "memory");
}
// shared -> global (tensor map, box at {x, y, z, slot}); elements outside the tensor are not written
__device__ __forceinline__ void tma_store_box(const CUtensorMap *map, int x, int y, int z, int slot, const void *src)
{
    asm volatile("cp.async.bulk.tensor.4d.global.shared::cta.bulk_group [%0, {%2, %3, %4, %5}], [%1];"
                 ::"l"(reinterpret_cast<uint64_t>(map)), "r"(smem_addr(src)), "r"(x), "r"(y), "r"(z), "r"(slot)
                 : "memory");
}
__device__ __forceinline__ void tma_store_commit_and_wait_read()
{
    asm volatile("cp.async.bulk.commit_group;" ::: "memory");
    asm volatile("cp.async.bulk.wait_group.read 0;" ::: "memory");
}
__device__ __forceinline__ void fence_proxy_async_smem()
{
    asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
}

// Where direction i of row y comes from (S1): the rules of load_dir.
struct Link {
    int slot, y, z;
    bool shifted;   // x is shifted by -c_x
};

template <int RM>
__device__ __forceinline__ Link tma_source(const KParams &p, int i, int y, int z)
{
    const int cy = TMA_CY[i], cz = TMA_CZ[i];
    Link l;
    if (RM == RD_LOCAL) {
        l.slot = i; l.y = y; l.z = z; l.shifted = false;
        return l;
    }
    const bool isbot = (y == 0), istop = (y == p.ny - 1);
    const bool bb = (cy == 1 && isbot && p.bot == BC_BOT_WALL) ||
                    (cy == -1 && istop && (p.top == BC_TOP_WALL || p.top == BC_TOP_LID));
    const bool fs = (cy == -1 && istop && p.top == BC_TOP_SLIP);
    const int s_n = (RM == RD_PULL) ? i : TMA_OPP[i];
    const int s_bb = (RM == RD_PULL) ? TMA_OPP[i] : i;
    const int s_fs = (RM == RD_PULL) ? TMA_MIR[i] : TMA_OPP[TMA_MIR[i]];
    int ys = y - cy;                                   // periodic wrap where the face is periodic
    if (ys < 0) ys = p.ny - 1;
    if (ys >= p.ny) ys = 0;
    int zs = z - cz;
    if (zs < 0) zs = p.nz - 1;
    if (zs >= p.nz) zs = 0;
    l.slot = bb ? s_bb : (fs ? s_fs : s_n);
    l.y = (bb || fs) ? y : ys;
    l.z = bb ? z : zs;
    l.shifted = !bb;
    return l;
}

template <int R> struct TmaOcc { static constexpr int minb = (R == 1) ? 8 : (R == 2 ? 4 : (R == 4 ? 2 : 1)); };

// grid = (nx/256) * (planes*ny/R) blocks, x chunks of a row adjacent (p.nchunk = nx/256);
// block = (64, R).  Dynamic shared memory: Q*R*256 floats (tile) + Q*R floats (halo words).
template <int RM, int WM, bool STATS, int R>
__global__ void __launch_bounds__(TMA_TX *R, TmaOcc<R>::minb)
step_tma_kernel(const KParams p, const __grid_constant__ CUtensorMap msrc)
{
    extern __shared__ __align__(128) unsigned char tma_smem[];
    float *buf = reinterpret_cast<float *>(tma_smem);   // [Q][R][256]
    float *halo = buf + Q * R * TMA_BOX;                 // [Q][R]
    __shared__ __align__(8) uint64_t bar;

    pdl_enter();
    const Ctx c = make_ctx<4>(p, p.z0 * p.ny);
    const int tx = threadIdx.x, ty = threadIdx.y, lin = ty * TMA_TX + tx;
    const int x0t = c.chunk * TMA_BOX;
    const int y0 = c.y - ty;                             // R | ny: the tile's rows share z

    if (lin == 0) mbar_init(&bar, 1);
    __syncthreads();

    // ---- S1: stream in.  Lane 0 of warp w moves the directions w, w + NW, ... (TMA instructions
    // take warp-uniform operands: one issuing lane per warp, all warps issue in parallel). ----
    constexpr int NW = (TMA_TX * R) / 32;
    const int warp = lin >> 5, lane = lin & 31;
    if (lin == 0) mbar_arrive_expect_tx(&bar, (uint32_t)(Q * R * TMA_BOX * 4));
    if (lane == 0) {
        for (int i = warp; i < Q; i += NW) {
#pragma unroll
            for (int r = 0; r < R; ++r) {
                const Link s = tma_source<RM>(p, i, y0 + r, c.z);
                tma_load_box(buf + (i * R + r) * TMA_BOX, &msrc, x0t, s.y, s.z, s.slot, &bar);
            }
        }
    }
    if (RM != RD_LOCAL) {
        // the element beyond the tile edge of every shifted box (periodic x wrap included)
        if (lin < Q * R) {
            const int i = lin / R, r = lin - i * R, cx = TMA_CX[i];
            const Link s = tma_source<RM>(p, i, y0 + r, c.z);
            if (s.shifted && cx != 0) {
                int xs = (cx == 1) ? x0t - 1 : x0t + TMA_BOX;
                xs = (xs < 0) ? p.nx - 1 : (xs >= p.nx ? 0 : xs);
                halo[lin] = p.src[(long long)s.slot * p.N + (long long)(s.y + p.ny * s.z) * p.nx + xs];
            }
        }
        __syncthreads();
    }
    const float cda = __ldg(p.cda + c.y);
    const float jr = __ldg(p.jref + c.y);
    mbar_wait(&bar, 0);

    // ---- read the thread's 4 cells x 19 directions back, x shift applied ----
    float g[Q][4];
    const float *mine = buf + ty * TMA_BOX + 4 * tx;
    static_for<0, Q>([&](auto ic) {
        constexpr int i = decltype(ic)::value;
        constexpr int cx = Lat::cx[i], cy = Lat::cy[i];
        const float *row = mine + i * R * TMA_BOX;
        const float4 t = *reinterpret_cast<const float4 *>(row);
        if constexpr (RM == RD_LOCAL || cx == 0) {
            g[i][0] = t.x; g[i][1] = t.y; g[i][2] = t.z; g[i][3] = t.w;
        } else {
            bool bb = false;                           // a bounce-back link reads the own cell: no shift
            if constexpr (cy == 1) bb = c.bot_bb;
            if constexpr (cy == -1) bb = c.top_bb;
            if constexpr (cx == 1) {                   // need x0-1 .. x0+2
                const float *nb = (tx == 0) ? halo + i * R + ty : row - 1;
                const float l = *nb;
                g[i][0] = bb ? t.x : l; g[i][1] = bb ? t.y : t.x; g[i][2] = bb ? t.z : t.y; g[i][3] = bb ? t.w : t.z;
            } else {                                   // need x0+1 .. x0+4
                const float *nb = (tx == TMA_TX - 1) ? halo + i * R + ty : row + 4;
                const float rr = *nb;
                g[i][0] = bb ? t.x : t.y; g[i][1] = bb ? t.y : t.z; g[i][2] = bb ? t.z : t.w; g[i][3] = bb ? t.w : rr;
            }
        }
        if constexpr (cy == -1) {
            if (c.top_lid) {
#pragma unroll
                for (int k = 0; k < 4; ++k) g[i][k] = p.lid[lid_index(i)];
            }
        }
    });

    // ---- S2-S8 as in step_kernel ----
    float s[NSTAT];
    cells_update<4, STATS, false, false>(p, g, s, cda, 0u, jr, 0ull, c.y);
    const Ctx c2 = (WM == WR_PUSH) ? make_ctx<4>(p, p.z0 * p.ny, true) : c;
    store_all<4, WM, false>(p, c2, g);
    if constexpr (STATS) {
        if (p.shift) {
            const float4 sh = __ldg(reinterpret_cast<const float4 *>(p.shift) + c2.y);
            stats_recentre(s, 4.0f, sh.x, sh.y, sh.z);
        }
        stats_row_reduce(p, c2, s);
    }
}

} // namespace lbm
