// lbm_tma_inst.cu — explicit instantiation of the TMA step launcher, selected by -DLBM_S=<0|1>
// (fused statistics): 9 kernels per translation unit (3 step kinds x 1, 2, 4 rows per tile).
#include "lbm_launch.cuh"
#include "lbm_tma.cuh"

#if !defined(LBM_S)
#error "compile with -DLBM_S=<0|1>"
#endif

namespace lbm {

template <int RM, int WM, bool S, int R>
static cudaError_t launch_tma_r(const StepLaunch &L, const KParams &p0)
{
    static bool attr_set = false;
    const int smem = (Q * R * TMA_BOX + Q * R) * 4;
    if (!attr_set) {
        cudaError_t e = cudaFuncSetAttribute(step_tma_kernel<RM, WM, S, R>, cudaFuncAttributeMaxDynamicSharedMemorySize, smem);
        if (e != cudaSuccess) return e;
        attr_set = true;
    }
    KParams p = p0;
    p.nchunk = L.nx / TMA_BOX;                   // tiles per row (make_ctx decomposes the block index with it)
    dim3 block(TMA_TX, R), grid((unsigned)((long long)(p.z1 - p.z0) * L.ny / R * p.nchunk));
    return launch_chain(step_tma_kernel<RM, WM, S, R>, grid, block, (size_t)smem, L.stream, L.pdl, p, *L.map);
}
template <int RM, int WM, bool S>
static cudaError_t launch_tma_rows(const StepLaunch &L, const KParams &p)
{
    switch (L.tma_rows) {
    case 4: return launch_tma_r<RM, WM, S, 4>(L, p);
    case 2: return launch_tma_r<RM, WM, S, 2>(L, p);
    default: return launch_tma_r<RM, WM, S, 1>(L, p);
    }
}

template <bool STATS>
cudaError_t launch_tma_t(const StepLaunch &L, const KParams &p)
{
    if (!L.aa) { if (L.tma_mode & 4) return launch_tma_rows<RD_PULL, WR_LOCAL, STATS>(L, p); }
    else if (!L.odd) { if (L.tma_mode & 1) return launch_tma_rows<RD_LOCAL, WR_LOCAL_OPP, STATS>(L, p); }
    else if (L.tma_mode & 2) return launch_tma_rows<RD_PULL_OPP, WR_PUSH, STATS>(L, p);
    return cudaErrorNotSupported;
}

template cudaError_t launch_tma_t<(LBM_S != 0)>(const StepLaunch &, const KParams &);

} // namespace lbm
