// kernels.h -- launch interface between api.cu and kernels.cu.
#pragma once
#include <cuda_runtime.h>

#include "device_mech.h"
#include "../../include/pyjac_b200.h"

namespace pyjac {

// device output pointers of one evaluation (NULL = skip)
struct EvalOut {
    double *rf, *rr, *cmod, *wdot;   // level 0
    double *dydt;                    // level 1
    double *jac;                     // level 2
    const double *v;                 // level 3: the vectors [n][ldv] (N_sp + 1 entries used per state)
    long long ldv;
    double *jv;                      // level 3: [n][N_sp + 1]
};

// level: 0 rates, 1 source term, 2 Jacobian, 3 Jacobian-vector product.  S: states a CTA interleaves per iteration (1, 2, 3, 4, 6);
// threads: a multiple of 32, at least 32 S, up to kMaxThreads.
const void *eval_kernel_ptr(int level, int S, bool stage);
size_t eval_smem_bytes(const SmemPlan &sp, int S);
cudaError_t launch_eval(int level, int threads, int S, const DeviceMech &m, const SmemPlan &sp, int grid, size_t smem,
                        long long n, const double *T, const double *P, const double *Y, long long ldy,
                        const EvalOut &out, cudaStream_t stream);

// adds to the count pyjac_kernel_launches() reports (kernels launched outside api.cu's `launch`)
void count_launches(int k);
// the device a handle's tables live on
int mech_device(const pyjac_mech *m);
// ... and the number of SMs of that device
int mech_sm_count(const pyjac_mech *m);

}  // namespace pyjac
