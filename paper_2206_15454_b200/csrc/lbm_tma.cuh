// lbm_tma.cuh — the fused step with the streaming done by the Tensor Memory Accelerator.
//
// Same time step as lbm::step_kernel (Algorithm 1; the per-cell arithmetic is
// the same moments()/collide() code), different data movement.  In step_kernel every thread moves
// its own 4 cells with 128-bit accesses and pays for the +-1 x shift of 10 of the 19 directions
// (Eq. 1) with shuffles, per-lane selects and scalar edge accesses: 13.8 warp instructions per
// cell on the AA odd step against 9.8 on the even one (profiles/r01_README.md).  Here a CTA owns a
// tile of 256 x R cells (R consecutive y rows of one z plane) and
//   1. 19 lanes of warp 0 (one per direction) issue `cp.async.bulk.tensor` loads of the tile's
//      R row segments of "their" population from wherever the streaming step says they come from:
//      the box start coordinate carries the shift (x0 - c_x, y - c_y, z - c_z, slot), so the
//      misalignment is absorbed by the TMA unit and the data lands ALIGNED in shared memory;
//      boundary links (bounce-back, free-slip, periodic y, z wrap) are only a different
//      (slot, y, z) of the box; all loads complete on one mbarrier;
//   2. every thread reads its 4 cells x 19 populations with 19 LDS.128, runs moments / drag /
//      Smagorinsky / collision (+ fused statistics), writes the result back to the same shared
//      memory words (19 STS.128);
//   3. after fence.proxy.async + one block barrier the 19 lanes issue `cp.async.bulk.tensor`
//      stores with the push coordinates (x0 + c_x, ...), commit, wait for the reads of shared
//      memory to finish and the CTA retires.  Several CTAs per SM overlap these phases.
// The periodic x wrap is the one thing a box cannot express (coordinate -1 / nx is out of bounds:
// loads fill zeros, stores clip): the issuing lane fetches / writes that single element of an
// edge tile with a plain scalar access.
//
// Requirements: 4 cells per thread layout (nx % 256 == 0), R | ny, no solid mask.  Everything
// else (AA even/odd, two-lattice pull, lid, slabs) goes through the same kernel.
#pragma once
#include <cuda.h>

#include "lbm_kernels.cuh"

namespace lbm {

constexpr int TMA_BOX = 256;              // cells of a row segment = one TMA box (hardware max 256)
constexpr int TMA_TX = TMA_BOX / 4;       // threads along x

__constant__ signed char TMA_CX[Q] = {0, 1, -1, 0, 0, 0, 0, 1, -1, 1, -1, 1, -1, 1, -1, 0, 0, 0, 0};
__constant__ signed char TMA_CY[Q] = {0, 0, 0, 1, -1, 0, 0, 1, -1, -1, 1, 0, 0, 0, 0, 1, -1, 1, -1};
__constant__ signed char TMA_CZ[Q] = {0, 0, 0, 0, 0, 1, -1, 0, 0, 0, 0, 1, -1, -1, 1, 1, -1, -1, 1};
__constant__ signed char TMA_OPP[Q] = {0, 2, 1, 4, 3, 6, 5, 8, 7, 10, 9, 12, 11, 14, 13, 16, 15, 18, 17};
__constant__ signed char TMA_MIR[Q] = {0, 1, 2, 4, 3, 5, 6, 9, 10, 7, 8, 11, 12, 13, 14, 18, 17, 16, 15};

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

// Where direction i of row y comes from (S1) / goes to (S7): the rules of load_dir / store_dir.
struct Link {
    int slot, y, z;
    bool shifted;   // x is shifted by -c_x (source) / +c_x (destination)
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

template <int WM>
__device__ __forceinline__ Link tma_dest(const KParams &p, int i, int y, int z)
{
    const int cy = TMA_CY[i], cz = TMA_CZ[i];
    Link l;
    if (WM != WR_PUSH) {
        l.slot = (WM == WR_LOCAL) ? i : TMA_OPP[i]; l.y = y; l.z = z; l.shifted = false;
        return l;
    }
    const bool isbot = (y == 0), istop = (y == p.ny - 1);
    const bool bb = (cy == -1 && isbot && p.bot == BC_BOT_WALL) ||
                    (cy == 1 && istop && (p.top == BC_TOP_WALL || p.top == BC_TOP_LID));
    const bool fs = (cy == 1 && istop && p.top == BC_TOP_SLIP);
    int yd = y + cy;
    if (yd < 0) yd = p.ny - 1;
    if (yd >= p.ny) yd = 0;
    int zd = z + cz;
    if (zd < 0) zd = p.nz - 1;
    if (zd >= p.nz) zd = 0;
    l.slot = bb ? TMA_OPP[i] : (fs ? TMA_MIR[i] : i);
    l.y = (bb || fs) ? y : yd;
    l.z = bb ? z : zd;
    l.shifted = !bb;
    return l;
}

template <int R> struct TmaOcc { static constexpr int minb = (R == 1) ? 8 : (R == 2 ? 4 : (R == 4 ? 2 : 1)); };

// grid = (nx/256) * (planes*ny/R) blocks, x chunks of a row adjacent; block = (64, R).
// Dynamic shared memory: Q*R*256 floats.
template <int RM, int WM, bool STATS, int R>
__global__ void __launch_bounds__(TMA_TX *R, TmaOcc<R>::minb)
step_tma_kernel(const KParams p, const __grid_constant__ CUtensorMap msrc, const __grid_constant__ CUtensorMap mdst)
{
    extern __shared__ __align__(128) unsigned char tma_smem[];
    float *buf = reinterpret_cast<float *>(tma_smem);   // [Q][R][256]
    __shared__ __align__(8) uint64_t bar;
    __shared__ float sred[STATS ? 2 * R : 1][NSTAT];

    const int tx = threadIdx.x, ty = threadIdx.y, lin = ty * TMA_TX + tx;
    const int nch = p.nx / TMA_BOX;
    const int rb = blockIdx.x / nch, chunk = blockIdx.x - rb * nch;
    const int x0t = chunk * TMA_BOX;
    const int row0 = p.z0 * p.ny + rb * R;
    const int z = row0 / p.ny, y0 = row0 - z * p.ny;
    const bool edge0 = (x0t == 0), edge1 = (x0t + TMA_BOX == p.nx);
    const bool xshift = (RM != RD_LOCAL) || (WM == WR_PUSH);

    if (lin == 0) mbar_init(&bar, 1);
    __syncthreads();

    // ---- S1: stream in.  Lane i of warp 0 moves direction i. ----
    float wrapv[R];
    if (lin < 32) {
        if (lin == 0) mbar_arrive_expect_tx(&bar, (uint32_t)(Q * R * TMA_BOX * 4));
        __syncwarp();
        if (lin < Q) {
            const int i = lin, cx = TMA_CX[i];
#pragma unroll
            for (int r = 0; r < R; ++r) {
                const Link s = tma_source<RM>(p, i, y0 + r, z);
                const int sx = s.shifted ? cx : 0;
                tma_load_box(buf + (i * R + r) * TMA_BOX, &msrc, x0t - sx, s.y, s.z, s.slot, &bar);
                wrapv[r] = 0.f;
                if (RM != RD_LOCAL) {
                    const float *rowp = p.src + (long long)s.slot * p.N + (long long)(s.y + p.ny * s.z) * p.nx;
                    if (sx == 1 && edge0) wrapv[r] = rowp[p.nx - 1];
                    if (sx == -1 && edge1) wrapv[r] = rowp[0];
                }
            }
        }
    }
    const int y = y0 + ty;
    const float cda = __ldg(p.cda + y);
    const float jr = __ldg(p.jref + y);
    mbar_wait(&bar, 0);
    if (RM != RD_LOCAL && (edge0 || edge1)) {
        // the element a box cannot reach: x = -1 / x = nx of the periodic row
        if (lin < Q) {
            const int i = lin, cx = TMA_CX[i];
#pragma unroll
            for (int r = 0; r < R; ++r) {
                const Link s = tma_source<RM>(p, i, y0 + r, z);
                if (s.shifted && cx == 1 && edge0) buf[(i * R + r) * TMA_BOX] = wrapv[r];
                if (s.shifted && cx == -1 && edge1) buf[(i * R + r) * TMA_BOX + TMA_BOX - 1] = wrapv[r];
            }
        }
        __syncthreads();
    }

    // ---- S2-S6 on the thread's 4 cells ----
    float g[Q][4];
    float *mine = buf + ty * TMA_BOX + 4 * tx;
    static_for<0, Q>([&](auto ic) {
        constexpr int i = decltype(ic)::value;
        const float4 t = *reinterpret_cast<const float4 *>(mine + i * R * TMA_BOX);
        g[i][0] = t.x; g[i][1] = t.y; g[i][2] = t.z; g[i][3] = t.w;
        if constexpr (Lat::cy[i] == -1) {
            if (p.top == BC_TOP_LID && y == p.ny - 1) {
#pragma unroll
                for (int k = 0; k < 4; ++k) g[i][k] = p.lid[lid_index(i)];
            }
        }
    });
    float s[NSTAT];
    if constexpr (STATS) {
#pragma unroll
        for (int k = 0; k < NSTAT; ++k) s[k] = 0.f;
    }
#pragma unroll
    for (int k = 0; k < 4; ++k) {
        mom_ref_shift<4>(g, k, jr);
        const Cell m = moments<4>(p, g, k, cda, jr);
        if constexpr (STATS) stats_add(s, m);
        collide<4>(p, g, k, m, jr);
    }
    static_for<0, Q>([&](auto ic) {
        constexpr int i = decltype(ic)::value;
        *reinterpret_cast<float4 *>(mine + i * R * TMA_BOX) = make_float4(g[i][0], g[i][1], g[i][2], g[i][3]);
    });
    fence_proxy_async_smem();

    // ---- S8: x-row sums of the statistics (two warps per row segment) ----
    float v4 = 0.f;
    bool owner = false;
    int col = 0;
    if constexpr (STATS) {
        if (p.shift) {
            const float4 sh = __ldg(reinterpret_cast<const float4 *>(p.shift) + y);
            stats_recentre(s, 4.0f, sh.x, sh.y, sh.z);
        }
        stats_warp_butterfly(s, lin & 31, v4, owner, col);
        if (owner) sred[lin >> 5][col] = v4;
    }
    __syncthreads();

    // ---- S7: stream out ----
    if (lin < Q) {
        const int i = lin, cx = TMA_CX[i];
#pragma unroll
        for (int r = 0; r < R; ++r) {
            const Link d = tma_dest<WM>(p, i, y0 + r, z);
            const int sx = d.shifted ? cx : 0;
            const float *srcp = buf + (i * R + r) * TMA_BOX;
            tma_store_box(&mdst, x0t + sx, d.y, d.z, d.slot, srcp);
            if (WM == WR_PUSH) {
                float *rowp = p.dst + (long long)d.slot * p.N + (long long)(d.y + p.ny * d.z) * p.nx;
                if (sx == 1 && edge1) rowp[0] = srcp[TMA_BOX - 1];
                if (sx == -1 && edge0) rowp[p.nx - 1] = srcp[0];
            }
        }
        tma_store_commit_and_wait_read();
    }
    if constexpr (STATS) {
        if (tx < NSTAT) {
            const long long pstride = (long long)p.nz * p.pchunks;
            float *out = p.partial + ((long long)y * NSTAT + tx) * pstride + (long long)z * p.pchunks + chunk;
            *out = sred[2 * ty][tx] + sred[2 * ty + 1][tx];
        }
    }
    (void)xshift;
}

} // namespace lbm
