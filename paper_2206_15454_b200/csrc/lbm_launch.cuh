// lbm_launch.cuh — launchers of the fused step kernel, one explicit instantiation per translation
// unit so that the ~130 step-kernel variants compile in parallel (build.py).
//
// lbm_api.cu fills a StepLaunch (the few handle fields a launch needs) and calls
// launch_step_t<V, STATS, SGS> / launch_tma_t<STATS>; lbm_step_inst.cu and lbm_tma_inst.cu hold the
// definitions, compiled once per (V, STATS, SGS) / (STATS).
#pragma once
#include <cuda.h>

#include "lbm_kernels.cuh"

namespace lbm {

constexpr int TMA_BOX = 256;   // cells of a row segment = one TMA box (hardware max 256)

struct StepLaunch {
    int TX, TY, nchunk;      // block shape and blocks per x row
    int nx, ny;
    bool mask;               // geometry handle (solid mask / forest codes)
    bool aa, aax;            // single-array storage (AA, x-balanced AA); neither: two-lattice
    bool odd;                // time parity of the state the step reads
    bool grid3;              // allow the 3-D grid form of the launch (A-B switch LBM_GRID3, default on)
    bool pdl;                // programmatic dependent launch (A-B switch LBM_PDL, default on)
    int tma_mode, tma_rows;  // TMA stream-in: step kinds (bit 0 AA even, 1 AA odd, 2 pull), rows per tile
    const CUtensorMap *map;  // tensor map of the array this step reads (TMA only)
    cudaStream_t stream;
};

// Kernel launch with the programmatic-stream-serialization attribute (programmatic dependent launch):
// the step kernels and the statistics stage 2 start with griddepcontrol.wait + launch_dependents
// (lbm_kernels.cuh: pdl_enter), so the NEXT launch of the chain is set up on the SMs while the last
// wave of this one is still running and starts the moment its predecessor has completed and flushed -
// the launch latency, which is what bounds lattices of a few 10^5 cells (cfg1: a 3 us kernel), hides.
template <class... KArgs, class... Args>
inline cudaError_t launch_chain(void (*kern)(KArgs...), dim3 grid, dim3 block, size_t smem, cudaStream_t st, bool pdl,
                                Args... args)
{
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = grid; cfg.blockDim = block; cfg.dynamicSmemBytes = smem; cfg.stream = st;
    cudaLaunchAttribute at[1];
    at[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
    at[0].val.programmaticStreamSerializationAllowed = 1;
    cfg.attrs = at; cfg.numAttrs = pdl ? 1 : 0;
    return cudaLaunchKernelEx(&cfg, kern, args...);
}

// One launch of step_kernel<V, RM, WM, STATS, MASK, SGS> for the planes [p.z0, p.z1).
template <int V, bool STATS, bool SGS>
cudaError_t launch_step_t(const StepLaunch &L, const KParams &p);

// One launch of step_tma_kernel<RM, WM, STATS, R>; cudaErrorNotSupported when this step kind is
// not on the TMA path (the caller then takes launch_step_t).
template <bool STATS>
cudaError_t launch_tma_t(const StepLaunch &L, const KParams &p);

#define LBM_DECLARE_STEP(V, S, G) \
    extern template cudaError_t launch_step_t<V, S, G>(const StepLaunch &, const KParams &);
LBM_DECLARE_STEP(4, false, false) LBM_DECLARE_STEP(4, true, false) LBM_DECLARE_STEP(4, false, true) LBM_DECLARE_STEP(4, true, true)
LBM_DECLARE_STEP(2, false, false) LBM_DECLARE_STEP(2, true, false) LBM_DECLARE_STEP(2, false, true) LBM_DECLARE_STEP(2, true, true)
LBM_DECLARE_STEP(1, false, false) LBM_DECLARE_STEP(1, true, false) LBM_DECLARE_STEP(1, false, true) LBM_DECLARE_STEP(1, true, true)
#undef LBM_DECLARE_STEP
extern template cudaError_t launch_tma_t<false>(const StepLaunch &, const KParams &);
extern template cudaError_t launch_tma_t<true>(const StepLaunch &, const KParams &);

} // namespace lbm
