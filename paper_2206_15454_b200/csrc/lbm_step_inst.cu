// lbm_step_inst.cu — one explicit instantiation of the step-kernel launcher, selected by
// -DLBM_V=<1|2|4> -DLBM_S=<0|1> -DLBM_G=<0|1> (cells per thread, fused statistics, row-table SGS):
// 10 kernels per translation unit (5 storage modes, each also as a geometry variant).  build.py compiles the
// twelve of them in parallel.
#include "lbm_launch.cuh"

#if !defined(LBM_V) || !defined(LBM_S) || !defined(LBM_G)
#error "compile with -DLBM_V=<1|2|4> -DLBM_S=<0|1> -DLBM_G=<0|1>"
#endif

namespace lbm {

template <int V, bool STATS, bool SGS>
cudaError_t launch_step_t(const StepLaunch &L, const KParams &p0)
{
    KParams p = p0;
    const int planes = p.z1 - p.z0;
    dim3 block(L.TX, L.TY), grid((unsigned)((long long)planes * L.ny / L.TY * L.nchunk));
    // block rows that divide ny: the 3-D grid with the same block order (make_ctx: no divisions)
    p.grid3 = (L.grid3 && L.ny % L.TY == 0 && L.ny / L.TY <= 65535 && planes <= 65535) ? 1 : 0;
    if (p.grid3) grid = dim3((unsigned)L.nchunk, (unsigned)(L.ny / L.TY), (unsigned)planes);
    cudaStream_t st = L.stream;
    if (L.mask) {
        if (!L.aa) return launch_chain(step_kernel<V, RD_PULL, WR_LOCAL, STATS, true, SGS>, grid, block, 0, st, L.pdl, p);
        else if (L.aax && !L.odd) return launch_chain(step_kernel<V, RD_XE, WR_XE, STATS, true, SGS>, grid, block, 0, st, L.pdl, p);
        else if (L.aax) return launch_chain(step_kernel<V, RD_XO, WR_XO, STATS, true, SGS>, grid, block, 0, st, L.pdl, p);
        else if (!L.odd) return launch_chain(step_kernel<V, RD_LOCAL, WR_LOCAL_OPP, STATS, true, SGS>, grid, block, 0, st, L.pdl, p);
        else return launch_chain(step_kernel<V, RD_PULL_OPP, WR_PUSH, STATS, true, SGS>, grid, block, 0, st, L.pdl, p);
    } else if (!L.aa) return launch_chain(step_kernel<V, RD_PULL, WR_LOCAL, STATS, false, SGS>, grid, block, 0, st, L.pdl, p);
    else if (L.aax && !L.odd) return launch_chain(step_kernel<V, RD_XE, WR_XE, STATS, false, SGS>, grid, block, 0, st, L.pdl, p);
    else if (L.aax) return launch_chain(step_kernel<V, RD_XO, WR_XO, STATS, false, SGS>, grid, block, 0, st, L.pdl, p);
    else if (!L.odd) return launch_chain(step_kernel<V, RD_LOCAL, WR_LOCAL_OPP, STATS, false, SGS>, grid, block, 0, st, L.pdl, p);
    else return launch_chain(step_kernel<V, RD_PULL_OPP, WR_PUSH, STATS, false, SGS>, grid, block, 0, st, L.pdl, p);
}

template cudaError_t launch_step_t<LBM_V, (LBM_S != 0), (LBM_G != 0)>(const StepLaunch &, const KParams &);

} // namespace lbm
