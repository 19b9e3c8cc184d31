// dispatch.cu -- switches over the (S, NP) shapes kernels.cu was compiled for (build.py: one object per shape).
#include "kernels.h"

namespace pyjac {

// (states per block, blocks per CTA iteration) -- keep in step with build.py
#define PYJAC_FOR_SHAPE(X) X(1, 1) X(1, 2) X(1, 3) X(1, 4) X(2, 1) X(2, 2) X(2, 3) X(2, 4)

#define PYJAC_DECL(SV, NPV)                                                                                         \
    const void *eval_kernel_ptr_##SV##_##NPV(int level);                                                           \
    cudaError_t launch_eval_##SV##_##NPV(int level, int threads, const DeviceMech &m, const SmemPlan &sp, int grid, \
                                         size_t smem, long long n, const double *T, const double *P,               \
                                         const double *Y, long long ldy, const EvalOut &out, cudaStream_t stream);
PYJAC_FOR_SHAPE(PYJAC_DECL)
#undef PYJAC_DECL

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

}  // namespace

cudaError_t launch_peak_store(double *buf, long long n_doubles, int grid, cudaStream_t stream)
{
    peak_store_kernel<<<grid, 256, 0, stream>>>(buf, n_doubles / 2);
    return cudaGetLastError();
}

cudaError_t launch_peak_dfma(double *out, long long iters, int grid, cudaStream_t stream)
{
    peak_dfma_kernel<<<grid, 256, 0, stream>>>(out, iters);
    return cudaGetLastError();
}

size_t eval_smem_bytes(const SmemPlan &sp, int S, int NP)
{
    return ((size_t)S * NP * sp.total + (size_t)sp.shared_total) * sizeof(double);
}

const void *eval_kernel_ptr(int level, int S, int NP)
{
#define PYJAC_PTR(SV, NPV) \
    if (S == SV && NP == NPV) return eval_kernel_ptr_##SV##_##NPV(level);
    PYJAC_FOR_SHAPE(PYJAC_PTR)
#undef PYJAC_PTR
    return nullptr;
}

cudaError_t launch_eval(int level, int threads, int S, int NP, const DeviceMech &m, const SmemPlan &sp, int grid,
                        size_t smem, long long n, const double *T, const double *P, const double *Y, long long ldy,
                        const EvalOut &out, cudaStream_t stream)
{
#define PYJAC_CASE(SV, NPV) \
    if (S == SV && NP == NPV) return launch_eval_##SV##_##NPV(level, threads, m, sp, grid, smem, n, T, P, Y, ldy, out, stream);
    PYJAC_FOR_SHAPE(PYJAC_CASE)
#undef PYJAC_CASE
    return cudaErrorInvalidValue;
}

}  // namespace pyjac
