// api.cu -- the C ABI of include/pyjac_b200.h: handle management, launches, host-buffer variants.
#include <cuda_runtime.h>

#include <atomic>
#include <cstdint>
#include <cstdlib>
#include <cstring>
#include <map>
#include <mutex>
#include <new>
#include <utility>
#include <vector>

#include "device_mech.h"
#include "kernels.h"
#include "mech_pack.h"

using namespace pyjac;

struct pyjac_mech {
    int device = 0;
    int ns = 0, nr = 0;
    void *blob = nullptr;       // one device allocation holding every table
    DeviceMech dm{};
    SmemPlan plan{};
    int threads = 128;
    int S = 1;                  // states per CTA iteration
    size_t smem[4] = {0, 0, 0, 0}; // dynamic shared memory per level
    int ctas_per_sm[4] = {1, 1, 1, 1};
    int n_sm = 1;
    // staging of the *_host calls: two device buffer pairs and two streams, kept between calls.  The handle
    // is otherwise immutable; this part is guarded by `ws_busy` (a caller that finds it taken stages with
    // temporary buffers instead).
    mutable std::atomic_flag ws_busy = ATOMIC_FLAG_INIT;
    mutable double *ws_in[2] = {nullptr, nullptr}, *ws_out[2] = {nullptr, nullptr};
    mutable size_t ws_in_cap = 0, ws_out_cap = 0;          // doubles per buffer
    mutable cudaStream_t ws_stream[2] = {nullptr, nullptr};
};

namespace {

std::atomic<long long> g_launches{0};

// reason of the last failed pyjac_mech_create* on this thread (static strings only), "" after a success
thread_local const char *t_last_error = "";

// preferred shared-memory carve-out (percent) set so far per (device, kernel function); see pyjac_mech_create_shaped
std::mutex g_carveout_mutex;
std::map<std::pair<int, const void *>, int> g_carveout;

struct Uploader {
    std::vector<unsigned char> host;
    std::vector<std::pair<const void **, size_t>> fix;   // (field, offset)
    template <class T>
    void add(const T **field, const std::vector<T> &v)
    {
        size_t off = (host.size() + 255) & ~size_t(255);
        host.resize(off + std::max<size_t>(v.size() * sizeof(T), 16));
        if (!v.empty()) std::memcpy(host.data() + off, v.data(), v.size() * sizeof(T));
        fix.push_back({(const void **)field, off});
    }
};

int check_eval_args(const pyjac_mech *m, int64_t n, const double *T, const double *P, const double *Y,
                    int64_t ldy)
{
    if (!m || n < 0) return PYJAC_EINVAL;
    if (n == 0) return PYJAC_OK;
    if (!T || !P || !Y || ldy < m->ns) return PYJAC_EINVAL;
    return PYJAC_OK;
}

int launch(const pyjac_mech *m, int level, int64_t n, const double *T, const double *P, const double *Y,
           int64_t ldy, const EvalOut &out, void *stream)
{
    if (n == 0) return PYJAC_OK;
    int dev = -1;
    if (cudaGetDevice(&dev) != cudaSuccess) return PYJAC_ECUDA;
    if (dev != m->device && cudaSetDevice(m->device) != cudaSuccess) return PYJAC_ECUDA;
    long long cap = (long long)m->n_sm * m->ctas_per_sm[level];
    const long long blocks = (n + m->S - 1) / m->S;
    int grid = (int)(blocks < cap ? blocks : cap);
    cudaError_t e = launch_eval(level, m->threads, m->S, m->dm, m->plan, grid, m->smem[level], n, T, P, Y, ldy,
                                out, (cudaStream_t)stream);
    if (dev != m->device) cudaSetDevice(dev);
    if (e != cudaSuccess) return PYJAC_ECUDA;
    g_launches.fetch_add(1, std::memory_order_relaxed);
    return PYJAC_OK;
}

}  // namespace

namespace pyjac {
void count_launches(int k) { g_launches.fetch_add(k, std::memory_order_relaxed); }
int mech_device(const pyjac_mech *m) { return m->device; }
int mech_sm_count(const pyjac_mech *m) { return m->n_sm; }
}  // namespace pyjac

extern "C" {

int pyjac_mech_create(const pyjac_mech_desc *d, int device, pyjac_mech **out)
{
    return pyjac_mech_create_shaped(d, device, nullptr, out);
}

int pyjac_mech_create_shaped(const pyjac_mech_desc *d, int device, const pyjac_launch_shape *shape, pyjac_mech **out)
{
    t_last_error = "";
    if (!out) { t_last_error = "the output handle pointer is NULL"; return PYJAC_EINVAL; }
    *out = nullptr;
    // validate and pack first (no CUDA call yet) with the architecture's shared-memory size; the
    // real device's limit is checked below
    HostPack hp;
    const char *why = nullptr;
    int rc = pack_mechanism(d, hp, hints_from_shape(shape, 227 * 1024), &why);
    if (rc != PYJAC_OK) { t_last_error = why ? why : ""; return rc; }
    int prev = -1;
    cudaDeviceProp prop{};
    if (cudaGetDevice(&prev) != cudaSuccess || cudaSetDevice(device) != cudaSuccess ||
        cudaGetDeviceProperties(&prop, device) != cudaSuccess) {
        cudaGetLastError();
        t_last_error = "no usable CUDA device with this index";
        return PYJAC_ECUDA;
    }
    pyjac_mech *m = new (std::nothrow) pyjac_mech();
    if (!m) { cudaSetDevice(prev); t_last_error = "host allocation failed"; return PYJAC_ENOMEM; }
    m->device = device;
    m->ns = hp.ns;
    m->nr = hp.nr;
    m->n_sm = prop.multiProcessorCount;
    m->threads = hp.threads;
    m->S = hp.S;
    DeviceMech &dm = m->dm;
    dm.ns = hp.ns; dm.nr = hp.nr; dm.ld = hp.ns + 1;
    dm.n_pd = hp.n_pd; dm.n_pk = hp.n_pk; dm.n_rchunk = hp.n_rchunk; dm.n_plain = (int)hp.n_plain_chunks;
    dm.n_arow = hp.n_arow; dm.n_arow01 = hp.n_arow01;
    dm.brk_common = hp.brk_common;
    dm.n_p1item = (int)hp.p1item.size();
    dm.rp = hp.rp; dm.n_slab = hp.n_slab;
    dm.eQ = hp.eQ; dm.eH = hp.eH; dm.eAlpha = hp.eAlpha; dm.eGamma = hp.eGamma; dm.eTc = hp.eTc;
    dm.eWdot = hp.eWdot; dm.eG0 = hp.eG0;
    dm.eS1 = hp.eS1; dm.eA0 = hp.eA0; dm.eS4 = hp.eS4; dm.eZero = hp.eZero; dm.eDump = hp.eDump; dm.eHs = hp.eHs;
    dm.n_e = hp.n_e;
    dm.n_aent = (int)(hp.a_ent.size() / 4); dm.n_bent = (int)(hp.b_ent.size() / 4); dm.n_achunk = (int)(hp.achunk.size() / 2);
    Uploader up;
    try {
        up.add(&dm.inv_mw, hp.inv_mw); up.add(&dm.mw, hp.mw);
        up.add(&dm.colc, hp.colc); up.add(&dm.wrow, hp.wrow);
        up.add(&dm.nasa, hp.nasa); up.add(&dm.t_mid, hp.t_mid);
        up.add((const uint32_t **)&dm.slots, hp.slots); up.add((const uint32_t **)&dm.vidx, hp.vidx);
        up.add(&dm.lnA, hp.lnA); up.add(&dm.beta, hp.beta); up.add(&dm.Ta, hp.Ta);
        up.add(&dm.rxn_orig, hp.rxn_orig); up.add(&dm.p1item, hp.p1item);
        up.add(&dm.rev_lnA, hp.rev_lnA); up.add(&dm.rev_beta, hp.rev_beta); up.add(&dm.rev_Ta, hp.rev_Ta);
        up.add(&dm.th_off, hp.th_off); up.add(&dm.th_data, hp.th_data); up.add(&dm.th_soa, hp.th_soa); up.add(&dm.th_brk, hp.th_brk);
        up.add(&dm.lo_lnA, hp.lo_lnA); up.add(&dm.lo_beta, hp.lo_beta); up.add(&dm.lo_Ta, hp.lo_Ta);
        up.add(&dm.fall_par, hp.fall_par);
        up.add(&dm.eff_base, hp.eff_base); up.add((const uint32_t **)&dm.eff_ent, hp.eff_ent);
        up.add(&dm.pk_ptr, hp.pk_ptr); up.add(&dm.pk_data, hp.pk_data);
        up.add((const uint32_t **)&dm.achunk, hp.achunk); up.add((const uint32_t **)&dm.a_ent, hp.a_ent);
        up.add((const uint32_t **)&dm.b_ent, hp.b_ent);
        up.add(&dm.bsplit, hp.bsplit);
    } catch (...) {
        delete m;
        cudaSetDevice(prev);
        t_last_error = "host allocation failed";
        return PYJAC_ENOMEM;
    }
    rc = PYJAC_OK;
    if (cudaMalloc(&m->blob, up.host.size()) != cudaSuccess) {
        rc = PYJAC_ENOMEM;
    } else if (cudaMemcpy(m->blob, up.host.data(), up.host.size(), cudaMemcpyHostToDevice) != cudaSuccess) {
        rc = PYJAC_ECUDA;
    }
    if (rc == PYJAC_OK) {
        for (auto &f : up.fix) *f.first = (const unsigned char *)m->blob + f.second;
        m->plan = hp.stage ? make_smem_plan(hp.ns, hp.n_e, (int)((hp.achunk.size() / 2 + 1) / 2), (int)(hp.a_ent.size() / 4),
                                            (int)(hp.b_ent.size() / 4))
                           : make_smem_plan(hp.ns, hp.n_e);
        const size_t bytes = eval_smem_bytes(m->plan, m->S);
        if (bytes + 64 > (size_t)prop.sharedMemPerBlockOptin || !eval_kernel_ptr(2, m->S, hp.stage)) {
            rc = PYJAC_ELIMIT;
        } else {
            // shared-memory carve-out: what the CTAs this shape was sized for need, the rest of the 256 KB
            // stays L1 (the gather tables are re-read from L1 / L2 by every CTA iteration)
            int carveout = (int)((100 * ((long long)hp.ctas_target * (long long)(bytes + 1024 + 16)) + 228 * 1024 - 1) / (228 * 1024));
            carveout = carveout > 100 ? 100 : carveout < 0 ? 0 : carveout;
            // The kernel functions are shared by every handle of this (S, stage): the carve-out of a function is
            // the LARGEST any handle on this device has asked for so far and is never lowered, so a handle made
            // later cannot take shared memory (and with it resident CTAs) away from an earlier one whose grid was
            // sized at its own creation; an earlier handle may at most find more CTAs resident than it counted.
            std::lock_guard<std::mutex> lock(g_carveout_mutex);
            for (int level = 0; level < 4 && rc == PYJAC_OK; ++level) {
                m->smem[level] = bytes;
                const void *k = eval_kernel_ptr(level, m->S, hp.stage);
                int &set = g_carveout[{device, k}];
                if (carveout < set) carveout = set;
                // the kernel function is shared by every handle of this shape: its dynamic shared-memory limit
                // is raised to what the device allows, once and for all, never to one handle's size
                cudaFuncAttributes fa{};
                if (cudaFuncGetAttributes(&fa, k) != cudaSuccess ||
                    cudaFuncSetAttribute(k, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                         (int)prop.sharedMemPerBlockOptin - (int)fa.sharedSizeBytes) != cudaSuccess ||
                    cudaFuncSetAttribute(k, cudaFuncAttributePreferredSharedMemoryCarveout, carveout) != cudaSuccess ||
                    cudaOccupancyMaxActiveBlocksPerMultiprocessor(&m->ctas_per_sm[level], k, m->threads, bytes) !=
                        cudaSuccess ||
                    m->ctas_per_sm[level] < 1)
                    rc = PYJAC_ECUDA;
                else
                    set = carveout;
            }
        }
    }
    cudaSetDevice(prev);
    if (rc != PYJAC_OK) {
        cudaGetLastError();
        if (m->blob) cudaFree(m->blob);
        delete m;
        t_last_error = rc == PYJAC_ELIMIT ? "the per-state tables of this launch shape exceed the device's shared memory per CTA"
                       : rc == PYJAC_ENOMEM ? "device allocation of the tables failed"
                                            : "a CUDA call failed while uploading the tables or configuring the kernels";
        return rc;
    }
    *out = m;
    return PYJAC_OK;
}

int pyjac_mech_destroy(pyjac_mech *m)
{
    if (!m) return PYJAC_OK;
    int prev = -1;
    cudaGetDevice(&prev);
    cudaSetDevice(m->device);
    cudaError_t e = cudaFree(m->blob);
    for (int b = 0; b < 2; ++b) {
        if (m->ws_stream[b]) cudaStreamDestroy(m->ws_stream[b]);
        if (m->ws_in[b]) cudaFree(m->ws_in[b]);
        if (m->ws_out[b]) cudaFree(m->ws_out[b]);
    }
    if (prev >= 0) cudaSetDevice(prev);
    delete m;
    return e == cudaSuccess ? PYJAC_OK : PYJAC_ECUDA;
}

int pyjac_mech_trim(pyjac_mech *m)
{
    if (!m) return PYJAC_EINVAL;
    if (m->ws_busy.test_and_set(std::memory_order_acquire)) return PYJAC_OK;      // a *_host call is using them: keep
    int prev = -1;
    cudaGetDevice(&prev);
    cudaError_t e = cudaSetDevice(m->device);
    for (int b = 0; b < 2 && e == cudaSuccess; ++b) {
        if (m->ws_in[b] && cudaFree(m->ws_in[b]) != cudaSuccess) e = cudaErrorUnknown;
        if (m->ws_out[b] && cudaFree(m->ws_out[b]) != cudaSuccess) e = cudaErrorUnknown;
        m->ws_in[b] = m->ws_out[b] = nullptr;
    }
    m->ws_in_cap = m->ws_out_cap = 0;
    if (prev >= 0) cudaSetDevice(prev);
    m->ws_busy.clear(std::memory_order_release);
    return e == cudaSuccess ? PYJAC_OK : PYJAC_ECUDA;
}

int pyjac_mech_sizes(const pyjac_mech *m, int32_t *ns, int32_t *nr)
{
    if (!m) return PYJAC_EINVAL;
    if (ns) *ns = m->ns;
    if (nr) *nr = m->nr;
    return PYJAC_OK;
}

int pyjac_eval_rates(const pyjac_mech *m, int64_t n, const double *T, const double *P, const double *Y,
                     int64_t ldy, double *rf, double *rr, double *cmod, double *wdot, void *stream)
{
    int rc = check_eval_args(m, n, T, P, Y, ldy);
    if (rc != PYJAC_OK) return rc;
    EvalOut out{rf, rr, cmod, wdot, nullptr, nullptr, nullptr, 0, nullptr};
    return launch(m, 0, n, T, P, Y, ldy, out, stream);
}

int pyjac_eval_dydt(const pyjac_mech *m, int64_t n, const double *T, const double *P, const double *Y,
                    int64_t ldy, double *dydt, void *stream)
{
    int rc = check_eval_args(m, n, T, P, Y, ldy);
    if (rc != PYJAC_OK) return rc;
    if (n > 0 && !dydt) return PYJAC_EINVAL;
    EvalOut out{nullptr, nullptr, nullptr, nullptr, dydt, nullptr, nullptr, 0, nullptr};
    return launch(m, 1, n, T, P, Y, ldy, out, stream);
}

int pyjac_eval_jacobian(const pyjac_mech *m, int64_t n, const double *T, const double *P, const double *Y,
                        int64_t ldy, double *jac, void *stream)
{
    int rc = check_eval_args(m, n, T, P, Y, ldy);
    if (rc != PYJAC_OK) return rc;
    if (n > 0 && !jac) return PYJAC_EINVAL;
    EvalOut out{nullptr, nullptr, nullptr, nullptr, nullptr, jac, nullptr, 0, nullptr};
    return launch(m, 2, n, T, P, Y, ldy, out, stream);
}

int pyjac_eval_jvp(const pyjac_mech *m, int64_t n, const double *T, const double *P, const double *Y,
                   int64_t ldy, const double *v, int64_t ldv, double *jv, void *stream)
{
    int rc = check_eval_args(m, n, T, P, Y, ldy);
    if (rc != PYJAC_OK) return rc;
    if (n > 0 && (!v || !jv || ldv < m->ns + 1)) return PYJAC_EINVAL;
    EvalOut out{nullptr, nullptr, nullptr, nullptr, nullptr, nullptr, v, (long long)ldv, jv};
    return launch(m, 3, n, T, P, Y, ldy, out, stream);
}

int64_t pyjac_kernel_launches(void) { return g_launches.load(std::memory_order_relaxed); }

int pyjac_jacobian_launch_config(const pyjac_mech *m, int64_t n, int32_t *threads, int32_t *smem_bytes,
                                 int32_t *ctas_per_sm, int32_t *grid, int32_t *states_per_cta)
{
    if (!m || n < 0) return PYJAC_EINVAL;
    if (threads) *threads = m->threads;
    if (states_per_cta) *states_per_cta = m->S;
    if (smem_bytes) *smem_bytes = (int32_t)m->smem[2];
    if (ctas_per_sm) *ctas_per_sm = m->ctas_per_sm[2];
    long long cap = (long long)m->n_sm * m->ctas_per_sm[2];
    const long long blocks = (n + m->S - 1) / m->S;
    if (grid) *grid = (int32_t)(blocks < cap ? blocks : cap);
    return PYJAC_OK;
}

const char *pyjac_mech_create_error(void) { return t_last_error; }

const char *pyjac_strerror(int code)
{
    switch (code) {
        case PYJAC_OK: return "success";
        case PYJAC_EINVAL: return "invalid argument or inconsistent mechanism description";
        case PYJAC_ENOMEM: return "host or device allocation failed";
        case PYJAC_ECUDA: return "CUDA runtime or launch error";
        case PYJAC_ELIMIT: return "mechanism exceeds a table limit of this build";
        case PYJAC_ESCRATCH:
            return "the call needs more scratch than the library's built-in 32 MiB device array holds "
                   "(pyjac_fd_static_max_states gives the largest batch)";
        default: return "unknown error code";
    }
}

}  // extern "C"

// ---- host-buffer variants: chunked, double-buffered H2D -> kernel -> D2H ---------------------------
namespace {

// largest staging buffer a handle keeps between *_host calls (two input and two output buffers: at most four times this,
// in practice ~2.1x because the inputs are small), and the size of the default chunk's output buffer
constexpr size_t kStageCacheBytes = (size_t)512 << 20;

int eval_host(const pyjac_mech *m, int level, int64_t n, const double *T, const double *P, const double *Y,
              int64_t ldy, double *outp, int64_t chunk_states)
{
    int rc = check_eval_args(m, n, T, P, Y, ldy);
    if (rc != PYJAC_OK) return rc;
    if (n == 0) return PYJAC_OK;
    if (!outp) return PYJAC_EINVAL;
    int prev = -1;
    if (cudaGetDevice(&prev) != cudaSuccess || cudaSetDevice(m->device) != cudaSuccess) return PYJAC_ECUDA;
    const int ns = m->ns, ld = ns + 1;
    const size_t out_per = level == 2 ? (size_t)ld * ld : (size_t)ld;
    const size_t in_per = (size_t)ns + 2;
    if (chunk_states <= 0) {
        size_t free_b = 0, total_b = 0;
        if (cudaMemGetInfo(&free_b, &total_b) != cudaSuccess) { cudaSetDevice(prev); return PYJAC_ECUDA; }
        const size_t per_state = (out_per + in_per) * sizeof(double) * 2;   // two buffers
        size_t c = (free_b / 4) / per_state;
        // by bytes, not by states: one output buffer of at most kStageCacheBytes (copies of that size already
        // overlap well; a 360-species Jacobian is 1 MB per state), so that what the handle keeps stays ~1 GiB
        const size_t want = kStageCacheBytes / ((out_per > in_per ? out_per : in_per) * sizeof(double));
        if (c > want) c = want;
        if (c < 1) c = 1;
        chunk_states = (int64_t)c;
    }
    if (chunk_states > n) chunk_states = n;
    const size_t C = (size_t)chunk_states;
    double *din[2] = {nullptr, nullptr}, *dout[2] = {nullptr, nullptr};
    cudaStream_t st[2] = {nullptr, nullptr};
    rc = PYJAC_OK;
    // the handle's staging buffers if nobody else is using them (grown on demand), else temporary ones
    // ... and only if the buffers are small enough to keep: a caller's explicit chunk beyond kStageCacheBytes per
    // buffer is staged through temporary buffers that are freed before the call returns
    const bool keepable = C * out_per * sizeof(double) <= kStageCacheBytes && C * in_per * sizeof(double) <= kStageCacheBytes;
    const bool cached = keepable && !m->ws_busy.test_and_set(std::memory_order_acquire);
    if (cached) {
        for (int b = 0; b < 2 && rc == PYJAC_OK; ++b)
            if (!m->ws_stream[b] && cudaStreamCreateWithFlags(&m->ws_stream[b], cudaStreamNonBlocking) != cudaSuccess)
                rc = PYJAC_ECUDA;
        if (rc == PYJAC_OK && (m->ws_in_cap < C * in_per || m->ws_out_cap < C * out_per)) {
            for (int b = 0; b < 2; ++b) {
                if (m->ws_in[b]) cudaFree(m->ws_in[b]);
                if (m->ws_out[b]) cudaFree(m->ws_out[b]);
                m->ws_in[b] = m->ws_out[b] = nullptr;
            }
            m->ws_in_cap = m->ws_out_cap = 0;
            for (int b = 0; b < 2 && rc == PYJAC_OK; ++b)
                if (cudaMalloc(&m->ws_in[b], C * in_per * sizeof(double)) != cudaSuccess ||
                    cudaMalloc(&m->ws_out[b], C * out_per * sizeof(double)) != cudaSuccess)
                    rc = PYJAC_ENOMEM;
            if (rc == PYJAC_OK) { m->ws_in_cap = C * in_per; m->ws_out_cap = C * out_per; }
        }
        for (int b = 0; b < 2; ++b) { din[b] = m->ws_in[b]; dout[b] = m->ws_out[b]; st[b] = m->ws_stream[b]; }
    } else {
        for (int b = 0; b < 2 && rc == PYJAC_OK; ++b) {
            if (cudaMalloc(&din[b], C * in_per * sizeof(double)) != cudaSuccess ||
                cudaMalloc(&dout[b], C * out_per * sizeof(double)) != cudaSuccess)
                rc = PYJAC_ENOMEM;
            else if (cudaStreamCreateWithFlags(&st[b], cudaStreamNonBlocking) != cudaSuccess)
                rc = PYJAC_ECUDA;
        }
    }
    int b = 0;
    for (int64_t s0 = 0; s0 < n && rc == PYJAC_OK; s0 += chunk_states, b ^= 1) {
        const size_t c = (size_t)((n - s0) < chunk_states ? (n - s0) : chunk_states);
        double *dT = din[b], *dP = din[b] + C, *dY = din[b] + 2 * C;
        cudaError_t e = cudaMemcpyAsync(dT, T + s0, c * sizeof(double), cudaMemcpyHostToDevice, st[b]);
        if (e == cudaSuccess) e = cudaMemcpyAsync(dP, P + s0, c * sizeof(double), cudaMemcpyHostToDevice, st[b]);
        if (e == cudaSuccess)
            e = cudaMemcpy2DAsync(dY, (size_t)ns * sizeof(double), Y + s0 * ldy, (size_t)ldy * sizeof(double),
                                  (size_t)ns * sizeof(double), c, cudaMemcpyHostToDevice, st[b]);
        if (e != cudaSuccess) { rc = PYJAC_ECUDA; break; }
        EvalOut out{nullptr, nullptr, nullptr, nullptr, level == 1 ? dout[b] : nullptr, level == 2 ? dout[b] : nullptr,
                    nullptr, 0, nullptr};
        rc = launch(m, level, (int64_t)c, dT, dP, dY, ns, out, st[b]);
        if (rc != PYJAC_OK) break;
        e = cudaMemcpyAsync(outp + (size_t)s0 * out_per, dout[b], c * out_per * sizeof(double),
                            cudaMemcpyDeviceToHost, st[b]);
        if (e != cudaSuccess) { rc = PYJAC_ECUDA; break; }
    }
    for (int q = 0; q < 2; ++q) {
        if (st[q] && cudaStreamSynchronize(st[q]) != cudaSuccess && rc == PYJAC_OK) rc = PYJAC_ECUDA;
        if (!cached) {
            if (st[q]) cudaStreamDestroy(st[q]);
            if (din[q]) cudaFree(din[q]);
            if (dout[q]) cudaFree(dout[q]);
        }
    }
    if (cached) m->ws_busy.clear(std::memory_order_release);
    if (rc != PYJAC_OK) cudaGetLastError();
    cudaSetDevice(prev);
    return rc;
}

}  // namespace

extern "C" {

int pyjac_eval_jacobian_host(const pyjac_mech *m, int64_t n, const double *T, const double *P, const double *Y,
                             int64_t ldy, double *jac, int64_t chunk_states)
{
    return eval_host(m, 2, n, T, P, Y, ldy, jac, chunk_states);
}

int pyjac_eval_dydt_host(const pyjac_mech *m, int64_t n, const double *T, const double *P, const double *Y,
                         int64_t ldy, double *dydt, int64_t chunk_states)
{
    return eval_host(m, 1, n, T, P, Y, ldy, dydt, chunk_states);
}

}  // extern "C"
