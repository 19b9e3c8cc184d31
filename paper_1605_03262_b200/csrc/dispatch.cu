// dispatch.cu -- switches over the S (states per CTA iteration) kernels.cu was compiled for (build.py: one object per S).
#include "kernels.h"

namespace pyjac {

// states a CTA interleaves per iteration -- keep in step with build.py
#define PYJAC_FOR_S(X) X(1) X(2) X(3) X(4) X(6)

#define PYJAC_DECL(SV)                                                                                             \
    const void *eval_kernel_ptr_##SV(int level, bool stage);                                                                   \
    cudaError_t launch_eval_##SV(int level, int threads, const DeviceMech &m, const SmemPlan &sp, int grid,        \
                                 size_t smem, long long n, const double *T, const double *P, const double *Y,      \
                                 long long ldy, const EvalOut &out, cudaStream_t stream);
PYJAC_FOR_S(PYJAC_DECL)
#undef PYJAC_DECL

size_t eval_smem_bytes(const SmemPlan &sp, int S) { return ((size_t)S * sp.total + (size_t)sp.shared_total) * sizeof(double); }

const void *eval_kernel_ptr(int level, int S, bool stage)
{
#define PYJAC_PTR(SV) \
    if (S == SV) return eval_kernel_ptr_##SV(level, stage);
    PYJAC_FOR_S(PYJAC_PTR)
#undef PYJAC_PTR
    return nullptr;
}

cudaError_t launch_eval(int level, int threads, int S, const DeviceMech &m, const SmemPlan &sp, int grid, size_t smem,
                        long long n, const double *T, const double *P, const double *Y, long long ldy,
                        const EvalOut &out, cudaStream_t stream)
{
#define PYJAC_CASE(SV) \
    if (S == SV) return launch_eval_##SV(level, threads, m, sp, grid, smem, n, T, P, Y, ldy, out, stream);
    PYJAC_FOR_S(PYJAC_CASE)
#undef PYJAC_CASE
    return cudaErrorInvalidValue;
}

}  // namespace pyjac
