// lbm_static.cu — the y-plane statistics of a (rho, u) field WITHOUT any allocation: the entry point
// lbm_plane_stats_static of include/lbm.h, for callers that cannot call cudaMalloc (code under CUDA
// graph capture, tight serving loops, harnesses that forbid it) and therefore cannot own the
// workspace a handle needs.
//
// What it computes is the two-stage reduction of the fused step (PAPER.md:L200,
// L251: averaging over time and over the homogeneous x-z planes) on ONE sample given as fields:
//   stage 1  x-row sums of u, v, w, uu, vv, ww, uv, vw, uw, rho of every (y, z) row -> scratch
//   stage 2  sum over z in fp64, then <a> and <a'b'> = <ab> - <a><b> per row y -> out[ny][10]
// (the columns of lbm_stats_read).  The handle path keeps the stage-1 partials in the caller-owned
// workspace; here they live in a file-scope device array of fixed size, LBM_STATIC_SCRATCH_BYTES,
// which every GPU that loads the library holds until the process exits.
//
// The array is shared by every call and keeps the last call's contents.  Nothing has to start at
// zero: stage 1 writes every entry stage 2 reads, stage 2 writes (does not accumulate) every output.
// Calls that overlap on the GPU (different streams, different threads) race on it.
#include "../../include/lbm.h"

#include <cuda_runtime.h>
#include <cstdio>
#include <mutex>

int lbm_fail_msg(int code, const char *msg);   // lbm_api.cu: sets the text of lbm_last_error()

namespace {

constexpr int NSTAT = 10;
constexpr int MAX_DEVICES = 64;

// the stage-1 partials: [y][k][z] floats, 10 * ny * nz * 4 bytes <= LBM_STATIC_SCRATCH_BYTES
static __device__ __align__(256) unsigned char g_scratch[LBM_STATIC_SCRATCH_BYTES];

// In host code `g_scratch` is a host-side stand-in, not a device address: the device address is
// looked up once per device, with that device current, and passed to the kernels.
float *g_scratch_dev[MAX_DEVICES];
std::mutex g_scratch_lock;

// Stage 1: block = 128 threads, one (y, z) row of nx cells; thread sums in fp64, warp shuffles,
// shared memory across the four warps, one fp32 partial per column.
__global__ void __launch_bounds__(128) plane_stage1_kernel(const float *__restrict__ rho, const float *__restrict__ u,
                                                           int nx, int ny, int nz, float *__restrict__ scratch)
{
    __shared__ double sm[4][NSTAT];
    const int y = blockIdx.x, z = blockIdx.y;
    const long long N = (long long)nx * ny * nz;
    const long long row = ((long long)z * ny + y) * nx;
    double s[NSTAT];
#pragma unroll
    for (int k = 0; k < NSTAT; ++k) s[k] = 0.0;
    for (int x = threadIdx.x; x < nx; x += blockDim.x) {
        const double a = u[row + x], b = u[N + row + x], c = u[2 * N + row + x];
        s[0] += a; s[1] += b; s[2] += c;
        s[3] += a * a; s[4] += b * b; s[5] += c * c;
        s[6] += a * b; s[7] += b * c; s[8] += a * c;
        s[9] += (double)rho[row + x];
    }
#pragma unroll
    for (int k = 0; k < NSTAT; ++k)
        for (int o = 16; o > 0; o >>= 1) s[k] += __shfl_xor_sync(0xffffffffu, s[k], o);
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    if (lane == 0) {
#pragma unroll
        for (int k = 0; k < NSTAT; ++k) sm[warp][k] = s[k];
    }
    __syncthreads();
    if (threadIdx.x < NSTAT) {
        const int k = threadIdx.x;
        const double t = (sm[0][k] + sm[1][k]) + (sm[2][k] + sm[3][k]);
        scratch[((long long)y * NSTAT + k) * nz + z] = (float)t;
    }
}

// Stage 2: one block per row y, warp k sums column k over z in fp64; thread 0 forms the statistics.
__global__ void __launch_bounds__(32 * NSTAT) plane_stage2_kernel(const float *__restrict__ scratch, int nz,
                                                                  double inv_count, double *__restrict__ out)
{
    __shared__ double tot[NSTAT];
    const int y = blockIdx.x, k = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const float *src = scratch + ((long long)y * NSTAT + k) * nz;
    double t = 0.0;
    for (int z = lane; z < nz; z += 32) t += (double)src[z];
    for (int o = 16; o > 0; o >>= 1) t += __shfl_xor_sync(0xffffffffu, t, o);
    if (lane == 0) tot[k] = t * inv_count;
    __syncthreads();
    if (threadIdx.x == 0) {
        double *r = out + (long long)y * NSTAT;
        const double mu = tot[0], mv = tot[1], mw = tot[2];
        r[0] = mu; r[1] = mv; r[2] = mw;
        r[3] = tot[3] - mu * mu; r[4] = tot[4] - mv * mv; r[5] = tot[5] - mw * mw;
        r[6] = tot[6] - mu * mv; r[7] = tot[7] - mv * mw; r[8] = tot[8] - mu * mw;
        r[9] = tot[9];
    }
}

int cuda_fail(const char *what, cudaError_t e)
{
    char msg[256];
    snprintf(msg, sizeof(msg), "lbm_plane_stats_static: %s failed: %s", what, cudaGetErrorString(e));
    return lbm_fail_msg(LBM_ECUDA, msg);
}

} // namespace

extern "C" int lbm_plane_stats_static(const float *rho_dev, const float *u_dev, int nx, int ny, int nz,
                                      double *out_dev, void *cuda_stream)
{
    if (nx < 1 || ny < 1 || nz < 1) return lbm_fail_msg(LBM_EINVAL, "lbm_plane_stats_static: lattice sizes must be >= 1");
    if ((double)nx * ny * nz >= 2147483648.0) return lbm_fail_msg(LBM_EINVAL, "lbm_plane_stats_static: nx*ny*nz must be < 2^31");
    if ((unsigned long long)ny * nz * NSTAT * sizeof(float) > (unsigned long long)LBM_STATIC_SCRATCH_BYTES || nz > 65535) {
        char msg[256];
        snprintf(msg, sizeof(msg),
                 "lbm_plane_stats_static: ny*nz = %lld rows need %lld bytes of scratch, the static array holds "
                 "%lld (ny*nz <= %lld, nz <= 65535); use a handle (lbm_stats_accumulate / lbm_stats_read) instead",
                 (long long)ny * nz, (long long)ny * nz * NSTAT * 4, (long long)LBM_STATIC_SCRATCH_BYTES,
                 (long long)(LBM_STATIC_SCRATCH_BYTES / (NSTAT * 4)));
        return lbm_fail_msg(LBM_EINVAL, msg);
    }
    if (!rho_dev || !u_dev || !out_dev) return lbm_fail_msg(LBM_EINVAL, "lbm_plane_stats_static: NULL pointer");
    cudaPointerAttributes at;
    cudaError_t e = cudaPointerGetAttributes(&at, rho_dev);
    if (e != cudaSuccess) return cuda_fail("cudaPointerGetAttributes", e);
    if (at.type != cudaMemoryTypeDevice && at.type != cudaMemoryTypeManaged)
        return lbm_fail_msg(LBM_EINVAL, "lbm_plane_stats_static: rho_dev is not device memory");
    const int dev = at.device;
    if (dev < 0 || dev >= MAX_DEVICES) return lbm_fail_msg(LBM_EINVAL, "lbm_plane_stats_static: device ordinal out of range");
    int prev = -1;
    if ((e = cudaGetDevice(&prev)) != cudaSuccess) return cuda_fail("cudaGetDevice", e);
    if (prev != dev && (e = cudaSetDevice(dev)) != cudaSuccess) return cuda_fail("cudaSetDevice", e);
    int rc = LBM_OK;
    float *scratch = nullptr;
    {
        // set-up, once per device, with that device current: the device address of the array
        std::lock_guard<std::mutex> lock(g_scratch_lock);
        if (!g_scratch_dev[dev]) {
            void *ptr = nullptr;
            e = cudaGetSymbolAddress(&ptr, g_scratch);
            if (e != cudaSuccess || !ptr) rc = cuda_fail("cudaGetSymbolAddress", e);
            else g_scratch_dev[dev] = static_cast<float *>(ptr);
        }
        scratch = g_scratch_dev[dev];
    }
    if (rc == LBM_OK) {
        cudaStream_t st = static_cast<cudaStream_t>(cuda_stream);
        plane_stage1_kernel<<<dim3((unsigned)ny, (unsigned)nz), 128, 0, st>>>(rho_dev, u_dev, nx, ny, nz, scratch);
        plane_stage2_kernel<<<(unsigned)ny, 32 * NSTAT, 0, st>>>(scratch, nz, 1.0 / ((double)nx * nz), out_dev);
        if ((e = cudaGetLastError()) != cudaSuccess) rc = cuda_fail("kernel launch", e);
    }
    if (prev != dev) cudaSetDevice(prev);
    return rc;
}
