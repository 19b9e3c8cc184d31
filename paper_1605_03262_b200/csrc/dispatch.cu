// dispatch.cu -- switches over the CTA sizes kernels.cu was compiled for (build.py: one object per size).
#include "kernels.h"

namespace pyjac {

// (threads per CTA, CTAs per SM the register budget is set for) -- keep in step with build.py
#define PYJAC_FOR_NT(X) X(128) X(256) X(384) X(512) X(768) X(1024)

#define PYJAC_DECL(N)                                                                                              \
    const void *eval_kernel_ptr_##N(int level, int S);                                                             \
    cudaError_t launch_eval_##N(int level, int S, const DeviceMech &m, const SmemPlan &sp, int grid, size_t smem,  \
                                long long n, const double *T, const double *P, const double *Y, long long ldy,     \
                                const EvalOut &out, cudaStream_t stream);
PYJAC_FOR_NT(PYJAC_DECL)
#undef PYJAC_DECL

size_t eval_smem_bytes(const SmemPlan &sp, int S) { return ((size_t)S * sp.total + (size_t)sp.shared_total) * sizeof(double); }

const void *eval_kernel_ptr(int level, int nt, int S)
{
#define PYJAC_PTR(N) \
    if (nt == N) return eval_kernel_ptr_##N(level, S);
    PYJAC_FOR_NT(PYJAC_PTR)
#undef PYJAC_PTR
    return nullptr;
}

cudaError_t launch_eval(int level, int nt, int S, const DeviceMech &m, const SmemPlan &sp, int grid, size_t smem,
                        long long n, const double *T, const double *P, const double *Y, long long ldy,
                        const EvalOut &out, cudaStream_t stream)
{
#define PYJAC_CASE(N) \
    if (nt == N) return launch_eval_##N(level, S, m, sp, grid, smem, n, T, P, Y, ldy, out, stream);
    PYJAC_FOR_NT(PYJAC_CASE)
#undef PYJAC_CASE
    return cudaErrorInvalidValue;
}

}  // namespace pyjac
