// tools.cu -- libpyjac_b200_tools.so: bench / test helpers of include/pyjac_b200_tools.h.  Not on the
// evaluation path: table statistics (host only) and the machine-peak probes.
#include <cuda_runtime.h>

#include "device_mech.h"
#include "mech_pack.h"
#include "../../include/pyjac_b200_tools.h"

using namespace pyjac;

namespace {

__global__ void __launch_bounds__(256) peak_store_kernel(double *buf, long long n_pairs)
{
    const long long stride = (long long)gridDim.x * blockDim.x;
    for (long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x; i < n_pairs; i += stride)
        asm volatile("st.global.cs.v2.f64 [%0], {%1, %2};" ::"l"(buf + 2 * i), "d"((double)i), "d"(1.0) : "memory");
}

__global__ void __launch_bounds__(256) peak_dfma_kernel(double *out, long long iters)
{
    const double x = 1.0 + 1e-9 * threadIdx.x, y = 1e-12 * blockIdx.x;
    double a0 = 0.1, a1 = 0.2, a2 = 0.3, a3 = 0.4, a4 = 0.5, a5 = 0.6, a6 = 0.7, a7 = 0.8;
    for (long long i = 0; i < iters; ++i) {
        a0 = fma(a0, x, y); a1 = fma(a1, x, y); a2 = fma(a2, x, y); a3 = fma(a3, x, y);
        a4 = fma(a4, x, y); a5 = fma(a5, x, y); a6 = fma(a6, x, y); a7 = fma(a7, x, y);
    }
    out[(long long)blockIdx.x * blockDim.x + threadIdx.x] = ((a0 + a1) + (a2 + a3)) + ((a4 + a5) + (a6 + a7));
}

// Tile probe: what a Jacobian kernel that assembles one state's matrix in shared memory and hands it to the bulk-copy
// engine would do for its output.  Per tile of `tile_doubles` doubles (one state's (N_s+1)^2 matrix): every element is
// written once with an 8-byte shared-memory store (MODE 0, 1: one STS.64 per element and lane, as a lane that owns a cell
// would), then either ONE cp.async.bulk.global.shared::cta of the whole tile issued by one thread (MODE 0: no load / store
// instruction of the SM touches the bytes again) or a read-back with LDS.128 and 16-byte streaming stores (MODE 1: the
// round-1 tile kernel's way, twice through the LSU data pipe).  Two tile buffers per CTA: the copy of tile t drains while
// tile t + 1 is filled.
template <int MODE>
__global__ void __launch_bounds__(256) peak_tile_store_kernel(double *out, long long n_tiles, int tile_doubles)
{
    extern __shared__ __align__(128) double tile_smem[];
    int buf = 0;
    for (long long t = blockIdx.x; t < n_tiles; t += gridDim.x, buf ^= 1) {
        double *b = tile_smem + (size_t)buf * tile_doubles;
        if (MODE == 0) {
            // this buffer went to the copy engine two tiles ago: wait until the engine has read it
            if (threadIdx.x == 0) asm volatile("cp.async.bulk.wait_group.read 1;" ::: "memory");
        }
        __syncthreads();
        for (int i = threadIdx.x; i < tile_doubles; i += blockDim.x) b[i] = (double)(t + i);
        if (MODE == 0) asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
        __syncthreads();
        double *g = out + t * (long long)tile_doubles;
        if (MODE == 0) {
            if (threadIdx.x == 0) {
                const unsigned src = (unsigned)__cvta_generic_to_shared(b);
                asm volatile("cp.async.bulk.global.shared::cta.bulk_group [%0], [%1], %2;" ::"l"(g), "r"(src),
                             "r"(tile_doubles * 8)
                             : "memory");
                asm volatile("cp.async.bulk.commit_group;" ::: "memory");
            }
        } else {
            for (int i = threadIdx.x; i < tile_doubles / 2; i += blockDim.x) {
                const double2 v = reinterpret_cast<const double2 *>(b)[i];
                asm volatile("st.global.cs.v2.f64 [%0], {%1, %2};" ::"l"(g + 2 * i), "d"(v.x), "d"(v.y) : "memory");
            }
        }
    }
    if (MODE == 0 && threadIdx.x == 0) asm volatile("cp.async.bulk.wait_group 0;" ::: "memory");
}

}  // namespace

extern "C" {

int pyjac_tools_pack_stats(const pyjac_mech_desc *d, const pyjac_launch_shape *shape, int64_t *stats)
{
    if (!stats) return PYJAC_EINVAL;
    HostPack hp;
    const int rc = pack_mechanism(d, hp, hints_from_shape(shape, 227 * 1024), nullptr);
    if (rc != PYJAC_OK) return rc;
    const SmemPlan plan = make_smem_plan(hp.ns, hp.n_e);
    for (int k = 0; k < PYJAC_TOOLS_NSTATS; ++k) stats[k] = 0;
    stats[0] = hp.n_e; stats[1] = hp.n_cell_entries; stats[2] = hp.n_b_steps; stats[3] = hp.n_a_steps;
    stats[4] = hp.n_cells; stats[5] = (int64_t)hp.achunk.size() / 2;
    stats[6] = (int64_t)(((size_t)hp.S * plan.total + (size_t)plan.shared_total) * sizeof(double));
    stats[7] = hp.n_rchunk; stats[8] = hp.S; stats[9] = hp.threads; stats[10] = 1; stats[11] = hp.ctas_target;
    stats[12] = hp.n_heavy_cells; stats[13] = hp.n_heavy_pieces; stats[14] = (int64_t)hp.a_ent.size() * 4;
    stats[15] = (int64_t)hp.b_ent.size() * 4;
    for (int k = 0; k < 4; ++k) stats[16 + k] = hp.n_a_steps_kind[k];
    stats[20] = hp.n_conflict_wf[0]; stats[21] = hp.n_conflict_wf[1];
    stats[22] = hp.n_layout_excess[0]; stats[23] = hp.n_layout_excess[1];
    return PYJAC_OK;
}

int pyjac_tools_peak_store_stream(double *buf, int64_t n_doubles, void *stream)
{
    if (!buf || n_doubles < 2 || (n_doubles & 1) || (reinterpret_cast<uintptr_t>(buf) & 15)) return PYJAC_EINVAL;
    int dev = 0, n_sm = 0;
    if (cudaGetDevice(&dev) != cudaSuccess ||
        cudaDeviceGetAttribute(&n_sm, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess)
        return PYJAC_ECUDA;
    peak_store_kernel<<<n_sm * 8, 256, 0, (cudaStream_t)stream>>>(buf, n_doubles / 2);
    return cudaGetLastError() == cudaSuccess ? PYJAC_OK : PYJAC_ECUDA;
}

int pyjac_tools_peak_tile_store(double *buf, int64_t n_tiles, int32_t tile_doubles, int32_t mode, int32_t ctas_per_sm,
                                void *stream)
{
    if (!buf || n_tiles < 1 || tile_doubles < 2 || (tile_doubles & 1) || (reinterpret_cast<uintptr_t>(buf) & 15) ||
        (mode != 0 && mode != 1) || ctas_per_sm < 1 || ctas_per_sm > 8)
        return PYJAC_EINVAL;
    const size_t smem = (size_t)2 * tile_doubles * sizeof(double);
    int dev = 0, n_sm = 0, optin = 0;
    if (cudaGetDevice(&dev) != cudaSuccess ||
        cudaDeviceGetAttribute(&n_sm, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess ||
        cudaDeviceGetAttribute(&optin, cudaDevAttrMaxSharedMemoryPerBlockOptin, dev) != cudaSuccess)
        return PYJAC_ECUDA;
    if (smem > (size_t)optin) return PYJAC_ELIMIT;
    auto k = mode == 0 ? peak_tile_store_kernel<0> : peak_tile_store_kernel<1>;
    if (cudaFuncSetAttribute(k, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem) != cudaSuccess) return PYJAC_ECUDA;
    k<<<n_sm * ctas_per_sm, 256, smem, (cudaStream_t)stream>>>(buf, n_tiles, tile_doubles);
    return cudaGetLastError() == cudaSuccess ? PYJAC_OK : PYJAC_ECUDA;
}

int pyjac_tools_peak_dfma(double *out, int64_t iters, int64_t *n_threads, void *stream)
{
    if (!out || iters < 1 || !n_threads) return PYJAC_EINVAL;
    int dev = 0, n_sm = 0;
    if (cudaGetDevice(&dev) != cudaSuccess ||
        cudaDeviceGetAttribute(&n_sm, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess)
        return PYJAC_ECUDA;
    *n_threads = (int64_t)n_sm * 2048;
    peak_dfma_kernel<<<n_sm * 8, 256, 0, (cudaStream_t)stream>>>(out, iters);
    return cudaGetLastError() == cudaSuccess ? PYJAC_OK : PYJAC_ECUDA;
}

}  // extern "C"
