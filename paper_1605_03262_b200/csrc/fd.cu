// fd.cu -- first-order forward-difference Jacobian built on the source-term kernel (Section 5.2:
// "a simple first-order forward difference adapted from CVODE", the paper's own comparison, Tables 4-5
// PAPER.md:823-853).  SURVEY.md section 8(f) row f2; the increment rule is DESIGN.md reading C21.
//
// Per state, with Phi = (T, Y_1 .. Y_{Ns-1}), N = N_s unknowns and f = dPhi/dt (pyjac_eval_dydt):
//   w_j    = 1 / (rtol |Phi_j| + atol)                        error weights
//   D_j    = max(sqrt(eps) |Phi_j|, sigma_0 / w_j)            increment of unknown j, sigma_0 = sqrt(eps)
//   J(:,j) = (f(Phi + D_j e_j) - f(Phi)) / D_j                 a mass-fraction increment is taken from Y_Ns (Eq. 2)
// (CVODE's sigma_0 = 1000 |h| eps N |f|_wrms carries the integrator's step h, which a stand-alone evaluation
// does not have.)
// Three steps per chunk of states: the source term of the states, one warp per state for the increments
// and the N perturbed states, the source term of those, and the difference quotient in the layout of
// pyjac_eval_jacobian (column N_s is zero).
#include <cuda_runtime.h>

#include <cstdint>
#include <mutex>

#include "kernels.h"

namespace {

constexpr double kSqrtEps = 1.4901161193847656e-08;

// one warp per state: increments inc[s][j] and the perturbed states (state s, unknown j) at row s * ns + j
__global__ void fd_perturb_kernel(int ns, long long n, const double *__restrict__ T, const double *__restrict__ P,
                                  const double *__restrict__ Y, long long ldy, double rtol, double atol, double *__restrict__ inc, double *__restrict__ Tp,
                                  double *__restrict__ Pp, double *__restrict__ Yp)
{
    const int lane = threadIdx.x & 31;
    const long long s = (long long)blockIdx.x * (blockDim.x >> 5) + (threadIdx.x >> 5);
    if (s >= n) return;
    const int last = ns - 1;
    const double *Ys = Y + s * ldy;
    const double Ts = T[s], Ps = P[s];
    for (int j = 0; j < ns; ++j) {
        const double phi = j == 0 ? Ts : Ys[j - 1];
        const double d = fmax(kSqrtEps * fabs(phi), kSqrtEps * (rtol * fabs(phi) + atol));
        const long long row = s * ns + j;
        if (lane == 0) {
            inc[row] = d;
            Tp[row] = j == 0 ? Ts + d : Ts;
            Pp[row] = Ps;
        }
        double *yp = Yp + row * ns;
        for (int k = lane; k < ns; k += 32) {
            double y = Ys[k];
            if (j > 0 && k == j - 1) y += d;
            if (j > 0 && k == last) y -= d;
            yp[k] = y;
        }
    }
}

// J[s][r + j ld] = (f1[s ns + j][r] - f0[s][r]) / inc[s][j]; column ns is zero
__global__ void fd_difference_kernel(int ns, long long n, const double *__restrict__ f0, const double *__restrict__ f1,
                                     const double *__restrict__ inc, double *__restrict__ jac)
{
    const int ld = ns + 1;
    const long long per = (long long)ld * ld;
    const long long total = n * per;
    for (long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x; i < total; i += (long long)gridDim.x * blockDim.x) {
        const long long s = i / per;
        const int e = (int)(i - s * per), j = e / ld, r = e - j * ld;
        double v = 0.0;
        if (j < ns) v = (f1[(s * ns + j) * ld + r] - f0[s * ld + r]) / inc[s * ns + j];
        __stcs(jac + i, v);
    }
}

}  // namespace

extern "C" {

int64_t pyjac_fd_workspace_doubles(const pyjac_mech *m, int64_t chunk_states)
{
    int32_t ns = 0;
    if (pyjac_mech_sizes(m, &ns, nullptr) != PYJAC_OK || chunk_states < 1) return -1;
    const int64_t ld = ns + 1;
    // f0, inc, perturbed T and P, perturbed Y, f1
    return chunk_states * (ld + (int64_t)ns + 2 * (int64_t)ns + (int64_t)ns * ns + (int64_t)ns * ld);
}

int pyjac_eval_jacobian_fd(const pyjac_mech *m, int64_t n, const double *T, const double *P, const double *Y,
                           int64_t ldy, double rtol, double atol, double *jac, double *work, int64_t work_doubles,
                           void *stream)
{
    int32_t ns = 0;
    if (pyjac_mech_sizes(m, &ns, nullptr) != PYJAC_OK || n < 0) return PYJAC_EINVAL;
    if (n == 0) return PYJAC_OK;
    if (!T || !P || !Y || !jac || !work || ldy < ns || !(rtol > 0.0) || !(atol > 0.0)) return PYJAC_EINVAL;
    const int64_t per_state = pyjac_fd_workspace_doubles(m, 1);
    int64_t chunk = work_doubles / per_state;
    if (chunk < 1) return PYJAC_EINVAL;
    if (chunk > n) chunk = n;
    const int64_t ld = ns + 1;
    double *f0 = work, *inc = f0 + chunk * ld, *Tp = inc + chunk * ns, *Pp = Tp + chunk * ns,
           *Yp = Pp + chunk * ns, *f1 = Yp + chunk * ns * ns;
    cudaStream_t st = (cudaStream_t)stream;
    int prev = -1;
    const int device = pyjac::mech_device(m);
    if (cudaGetDevice(&prev) != cudaSuccess) return PYJAC_ECUDA;
    if (prev != device && cudaSetDevice(device) != cudaSuccess) return PYJAC_ECUDA;
    int result = PYJAC_OK;
    const long long max_blocks = (long long)pyjac::mech_sm_count(m) * 16;      // grid-stride loop: 16 CTAs of 256 per SM
    for (int64_t s0 = 0; s0 < n && result == PYJAC_OK; s0 += chunk) {
        const int64_t c = n - s0 < chunk ? n - s0 : chunk;
        int rc = pyjac_eval_dydt(m, c, T + s0, P + s0, Y + s0 * ldy, ldy, f0, stream);
        if (rc != PYJAC_OK) { result = rc; break; }
        const int warps = 8;
        fd_perturb_kernel<<<(unsigned)((c + warps - 1) / warps), 32 * warps, 0, st>>>(
            ns, c, T + s0, P + s0, Y + s0 * ldy, ldy, rtol, atol, inc, Tp, Pp, Yp);
        if (cudaGetLastError() != cudaSuccess) { result = PYJAC_ECUDA; break; }
        pyjac::count_launches(1);
        rc = pyjac_eval_dydt(m, c * ns, Tp, Pp, Yp, ns, f1, stream);
        if (rc != PYJAC_OK) { result = rc; break; }
        const long long total = (long long)c * ld * ld;
        const long long blocks = (total + 255) / 256;
        fd_difference_kernel<<<(unsigned)(blocks < max_blocks ? blocks : max_blocks), 256, 0, st>>>(
            ns, c, f0, f1, inc, jac + s0 * ld * ld);
        if (cudaGetLastError() != cudaSuccess) { result = PYJAC_ECUDA; break; }
        pyjac::count_launches(1);
    }
    if (prev != device) cudaSetDevice(prev);
    return result;
}

}  // extern "C"

// ---- forward-difference Jacobian for callers that cannot allocate device memory -------------------------------
//
// pyjac_eval_jacobian_fd needs a caller-owned scratch buffer.  Some callers have no way to get one: a reacting-flow
// solver that handed the whole GPU to its own arena at start-up (a later cudaMalloc simply fails), an integrator
// callback that runs inside a time-step loop where cudaMalloc / cudaFree would stall every stream of the device
// through their device-wide synchronisation, or a plug-in whose host application forbids driver allocations after
// initialisation.  For them the scratch lives in the library image itself: a file-scope __device__ array of
// kFdStaticDoubles doubles (32 MiB), which every GPU that loads this library holds from module load to process exit.
//
// `g_fd_static_scratch` below is two different things.  In device code it is the array.  In host code the name is only
// a host-side shadow symbol: its host address is NOT device memory, and a kernel handed `g_fd_static_scratch` from
// the host would fault (or, on a system where the GPU can reach host memory, silently use the wrong bytes).  The
// host side therefore asks the runtime for the real device address, once per device, with that device current
// (fd_static_device_ptr), and passes that pointer to the kernels.
constexpr int64_t kFdStaticDoubles = (int64_t)4 << 20;        // 4 Mi doubles = 32 MiB per GPU
constexpr int kFdStaticMaxDevices = 64;

static __device__ __align__(256) double g_fd_static_scratch[kFdStaticDoubles];

namespace {

std::mutex g_fd_static_mutex;
double *g_fd_static_ptr[kFdStaticMaxDevices] = {};           // device address of the array, per device (NULL: not asked yet)

// Device address of g_fd_static_scratch on `device` (NULL on error).  The first call for a device makes that device
// current, resolves the symbol (which loads this module on the device if it is not loaded yet) and restores the
// caller's device; later calls return the cached pointer.
double *fd_static_device_ptr(int device)
{
    if (device < 0 || device >= kFdStaticMaxDevices) return nullptr;
    std::lock_guard<std::mutex> lock(g_fd_static_mutex);
    if (g_fd_static_ptr[device]) return g_fd_static_ptr[device];
    int prev = -1;
    if (cudaGetDevice(&prev) != cudaSuccess) return nullptr;
    if (prev != device && cudaSetDevice(device) != cudaSuccess) return nullptr;
    double *ptr = nullptr;
    const cudaError_t e = cudaGetSymbolAddress((void **)&ptr, g_fd_static_scratch);
    if (prev != device) cudaSetDevice(prev);
    if (e != cudaSuccess || !ptr) return nullptr;
    g_fd_static_ptr[device] = ptr;
    return ptr;
}

}  // namespace

extern "C" {

int64_t pyjac_fd_static_max_states(const pyjac_mech *m)
{
    const int64_t per_state = pyjac_fd_workspace_doubles(m, 1);
    if (per_state < 1) return -1;
    return kFdStaticDoubles / per_state;
}

int pyjac_eval_jacobian_fd_static(const pyjac_mech *m, int64_t n, const double *T, const double *P, const double *Y,
                                  int64_t ldy, double rtol, double atol, double *jac, void *stream)
{
    int32_t ns = 0;
    if (pyjac_mech_sizes(m, &ns, nullptr) != PYJAC_OK || n < 0) return PYJAC_EINVAL;
    if (n == 0) return PYJAC_OK;
    // one chunk only: the states of a call must fit the array together, the caller loops over larger batches
    if (n > pyjac_fd_static_max_states(m)) return PYJAC_ESCRATCH;
    double *scratch = fd_static_device_ptr(pyjac::mech_device(m));
    if (!scratch) return PYJAC_ECUDA;
    // Every scratch word a kernel of this path reads has been written earlier in the same call (f0 and f1 by the
    // source-term launches, the increments and perturbed states by fd_perturb_kernel), so what the previous call
    // left in the array is never seen and nothing has to be cleared.
    return pyjac_eval_jacobian_fd(m, n, T, P, Y, ldy, rtol, atol, jac, scratch, kFdStaticDoubles, stream);
}

}  // extern "C"
