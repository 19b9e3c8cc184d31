// tools.cu -- libpyjac_b200_tools.so: bench / test helpers of include/pyjac_b200_tools.h.  Not on the
// evaluation path: table statistics (host only) and the machine-peak probes.
#include <cuda_runtime.h>

#include <algorithm>
#include <cstdint>
#include <vector>

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

// Gather probe: a timing prototype of the output half of a Jacobian kernel WITHOUT padded gathers (round-2 verdict, item 1).
// It is not the evaluation: the per-reaction terms E of a state are stand-in values written once per CTA; what is real are
// the contribution lists of the Jacobian cells (HostPack::raw_cells of the mechanism: which E elements each cell sums, with
// which integer coefficient), their number and their length distribution.  Per batch of S states a CTA
//   (1) dense pass: every cell starts from the rank-one part alpha_r u_c - gamma_r v_c (a lane keeps its rows' alpha, gamma
//       in registers, u_c and v_c are warp-uniform loads) and is written to the state's tile in shared memory;
//   (2) sparse pass: the non-empty cells, sorted by list length and dealt out in chunks of 32 cells of (nearly) equal length,
//       one cell per lane: 4-byte entries (E index, coefficient) from global memory, one shared-memory load of E per entry
//       and state (the S states of an element are adjacent), the sum added to the cell in the tile;
//   (3) one cp.async.bulk per state moves the finished tile to global memory.
// n_buf = 2 tile sets let the copies of batch b drain while batch b + 1 is computed.
template <int S>
__global__ void __launch_bounds__(512) gather_probe_kernel(const uint32_t *__restrict__ ent, const uint32_t *__restrict__ chunk_hdr,
                                                           const uint16_t *__restrict__ cpos, int n_chunks, int n_e, int ld,
                                                           int e_alpha, int e_gamma, int n_buf, long long n_states,
                                                           double *__restrict__ out)
{
    extern __shared__ __align__(128) double probe_smem[];
    const int cells = ld * ld;
    double *E = probe_smem;                                    // [n_e][S]
    double *tiles = probe_smem + (((size_t)n_e * S + 15) & ~(size_t)15);   // [n_buf][S][cells]
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5, nw = blockDim.x >> 5;
    for (int i = threadIdx.x; i < n_e * S; i += blockDim.x) E[i] = 1.0 / (double)(1 + (i / S) % 1021);
    __syncthreads();
    const long long n_batches = (n_states + S - 1) / S;
    int buf = 0;
    for (long long b = blockIdx.x; b < n_batches; b += gridDim.x, buf = (buf + 1 == n_buf ? 0 : buf + 1)) {
        double *tile = tiles + (size_t)buf * S * cells;
        // the copies that last read this tile set must have finished reading it
        if (threadIdx.x == 0) {
            if (n_buf == 2) asm volatile("cp.async.bulk.wait_group.read 1;" ::: "memory");
            else asm volatile("cp.async.bulk.wait_group.read 0;" ::: "memory");
        }
        __syncthreads();
        // (1) dense pass: warp w takes columns w, w + nw, ..; lane takes rows lane, lane + 32, ..
        for (int r0 = 0; r0 < ld; r0 += 32) {
            const int r = r0 + lane;
            double al[S], ga[S];
#pragma unroll
            for (int q = 0; q < S; ++q) {
                al[q] = r < ld ? E[(size_t)(e_alpha + r) * S + q] : 0.0;
                ga[q] = r < ld ? E[(size_t)(e_gamma + r) * S + q] : 0.0;
            }
            for (int c = warp; c < ld; c += nw) {
#pragma unroll
                for (int q = 0; q < S; ++q) {
                    const double u = E[(size_t)c * S + q], v = E[(size_t)(ld + c) * S + q];
                    if (r < ld) tile[(size_t)q * cells + r + c * ld] = al[q] * u - ga[q] * v;
                }
            }
        }
        __syncthreads();
        // (2) sparse pass: chunk k of 32 cells, hdr = first entry row | steps << 24
        for (int k = warp; k < n_chunks; k += nw) {
            const uint32_t hdr = chunk_hdr[k];
            const int steps = (int)(hdr >> 24);
            const uint32_t *e = ent + (size_t)(hdr & 0xffffffu) * 32 + lane;
            const unsigned pos = cpos[(size_t)k * 32 + lane];
            double acc[S];
#pragma unroll
            for (int q = 0; q < S; ++q) acc[q] = 0.0;
#pragma unroll 4
            for (int st = 0; st < steps; ++st) {
                const uint32_t w = e[(size_t)st * 32];
                const double cf = (double)((int)(w & 255u) - 128);
                const double *src = E + (size_t)(w >> 8) * S;
#pragma unroll
                for (int q = 0; q < S; ++q) acc[q] = fma(cf, src[q], acc[q]);
            }
            if (pos != 0xffffu) {
#pragma unroll
                for (int q = 0; q < S; ++q) tile[(size_t)q * cells + pos] += acc[q];
            }
        }
        asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
        __syncthreads();
        // (3) one bulk copy per state
        if (threadIdx.x == 0) {
            for (int q = 0; q < S; ++q) {
                const long long state = b * S + q;
                if (state >= n_states) break;
                const unsigned src = (unsigned)__cvta_generic_to_shared(tile + (size_t)q * cells);
                asm volatile("cp.async.bulk.global.shared::cta.bulk_group [%0], [%1], %2;" ::"l"(out + state * cells), "r"(src),
                             "r"(cells * 8)
                             : "memory");
            }
            asm volatile("cp.async.bulk.commit_group;" ::: "memory");
        }
    }
    if (threadIdx.x == 0) asm volatile("cp.async.bulk.wait_group 0;" ::: "memory");
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

int pyjac_tools_gather_probe(const pyjac_mech_desc *d, int32_t S, int32_t threads, int32_t ctas_per_sm, int32_t n_buf,
                             int64_t n_states, double *out, double *expected_host, int64_t *stats, int32_t reps,
                             float *ms_best, float *ms_mean, void *stream)
{
    if (!d || !out || !expected_host || !stats || !ms_best || !ms_mean || n_states < 1 || reps < 1 || (S != 1 && S != 2 && S != 3) ||
        threads < 32 || threads > 512 || threads % 32 || ctas_per_sm < 1 || ctas_per_sm > 4 || (n_buf != 1 && n_buf != 2))
        return PYJAC_EINVAL;
    HostPack hp;
    ShapeHints hints = hints_from_shape(nullptr, 227 * 1024);
    hints.keep_cells = 1;
    hints.S = 1;                      // the tables of the evaluation kernel are not used here; any shape that packs will do
    int rc = pack_mechanism(d, hp, hints, nullptr);
    if (rc != PYJAC_OK) return rc;
    const int ld = hp.ns + 1, cells = ld * ld, n_e = hp.n_e;
    if (cells > 0xfffe || (cells * 8) % 16 != 0 || 2 * ld > n_e) return PYJAC_ELIMIT;
    // non-empty cells sorted by list length (longest first), 32 per chunk, padded to the chunk's longest list
    // Within one list length the cells are dealt out so that sixteen consecutive ones sit in sixteen different bank
    // pairs of the tile (their read-modify-write is then conflict-free while every bank pair still has a cell left).
    std::vector<int> order;
    {
        size_t longest = 0;
        for (int f = 0; f < cells; ++f) longest = std::max(longest, hp.raw_cells[(size_t)f].size());
        for (size_t len = longest; len >= 1; --len) {
            std::vector<std::vector<int>> bucket(16);
            size_t left = 0;
            for (int f = 0; f < cells; ++f)
                if (hp.raw_cells[(size_t)f].size() == len) { bucket[(size_t)f % 16].push_back(f); ++left; }
            for (size_t b = 0; left > 0; b = (b + 1) % 16)
                if (!bucket[b].empty()) { order.push_back(bucket[b].back()); bucket[b].pop_back(); --left; }
        }
    }
    std::vector<uint32_t> ent, hdr;
    std::vector<uint16_t> cpos;
    long long n_entries = 0;
    auto val = [&](uint32_t e) { return 1.0 / (double)(1 + e % 1021); };
    for (int r = 0; r < ld; ++r)
        for (int c = 0; c < ld; ++c)
            expected_host[r + c * ld] = val((uint32_t)(hp.eAlpha + r)) * val((uint32_t)c) - val((uint32_t)(hp.eGamma + r)) * val((uint32_t)(ld + c));
    for (size_t at = 0; at < order.size(); at += 32) {
        const size_t n = std::min<size_t>(32, order.size() - at);
        const size_t steps = hp.raw_cells[(size_t)order[at]].size();
        if (steps > 255 || ent.size() / 32 > 0xffffffu) return PYJAC_ELIMIT;
        hdr.push_back((uint32_t)(ent.size() / 32) | (uint32_t)steps << 24);
        const size_t base = ent.size();
        ent.resize(base + steps * 32, 128u);                       // padding: element 0 with coefficient 0
        std::vector<std::vector<std::pair<uint32_t, int>>> rest(32);      // entries not yet given a step, per lane
        for (size_t l = 0; l < 32; ++l) {
            if (l >= n) { cpos.push_back(0xffffu); continue; }
            const int f = order[at + l];
            cpos.push_back((uint16_t)f);
            rest[l] = hp.raw_cells[(size_t)f];
            for (auto &e : rest[l]) {
                if (e.second < -128 || e.second > 127 || e.first >= (uint32_t)n_e) return PYJAC_ELIMIT;
                expected_host[f] += (double)e.second * val(e.first);
            }
            n_entries += (long long)rest[l].size();
        }
        // The order of a lane's entries is free: step by step and half warp by half warp (the sixteen lanes of one
        // shared-memory wavefront of an 8-byte load), every lane takes the entry whose bank pair (E index mod 16; the S
        // states of an element are adjacent and S is 1, 2 or 3) is wanted least so far; lanes that have run out read a
        // zero-coefficient element of a bank pair nobody wants.  Greedy, not the exact edge colouring of mech_pack.cu.
        for (size_t st = 0; st < steps; ++st)
            for (size_t half = 0; half < 2; ++half) {
                int used[16] = {0};
                // lanes with the fewest choices first
                std::vector<size_t> lanes;
                for (size_t l = half * 16; l < half * 16 + 16; ++l) lanes.push_back(l);
                std::stable_sort(lanes.begin(), lanes.end(), [&](size_t a, size_t b) { return rest[a].size() < rest[b].size(); });
                for (size_t l : lanes) {
                    if (rest[l].empty()) continue;
                    // a lane must place all its entries in the steps that are left
                    size_t pick = 0;
                    for (size_t q = 1; q < rest[l].size(); ++q)
                        if (used[rest[l][q].first % 16] < used[rest[l][pick].first % 16]) pick = q;
                    if (rest[l].size() < steps - st && used[rest[l][pick].first % 16] > 0) continue;   // wait for a better step
                    ent[base + st * 32 + l] = rest[l][pick].first << 8 | (uint32_t)(rest[l][pick].second + 128);
                    used[rest[l][pick].first % 16] += 1;
                    rest[l].erase(rest[l].begin() + (long)pick);
                }
                for (size_t l = half * 16; l < half * 16 + 16; ++l)
                    if (ent[base + st * 32 + l] == 128u) {                 // padding: the least wanted bank pair
                        int b = 0;
                        for (int q = 1; q < 16; ++q)
                            if (used[q] < used[b]) b = q;
                        ent[base + st * 32 + l] = (uint32_t)b << 8 | 128u;
                        used[b] += 1;
                    }
            }
        for (size_t l = 0; l < 32; ++l)
            if (!rest[l].empty()) return PYJAC_ELIMIT;                     // cannot happen: a lane waits only while steps remain
    }
    const size_t smem = ((((size_t)n_e * S + 15) & ~(size_t)15) + (size_t)n_buf * S * cells) * sizeof(double);
    stats[0] = n_entries; stats[1] = (int64_t)ent.size(); stats[2] = (int64_t)hdr.size(); stats[3] = n_e;
    stats[4] = (int64_t)smem; stats[5] = (int64_t)order.size(); stats[6] = cells; stats[7] = 0;
    int dev = 0, n_sm = 0, optin = 0;
    if (cudaGetDevice(&dev) != cudaSuccess ||
        cudaDeviceGetAttribute(&n_sm, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess ||
        cudaDeviceGetAttribute(&optin, cudaDevAttrMaxSharedMemoryPerBlockOptin, dev) != cudaSuccess)
        return PYJAC_ECUDA;
    if (smem > (size_t)optin) return PYJAC_ELIMIT;
    auto k = S == 1 ? gather_probe_kernel<1> : S == 2 ? gather_probe_kernel<2> : gather_probe_kernel<3>;
    uint32_t *d_ent = nullptr, *d_hdr = nullptr;
    uint16_t *d_pos = nullptr;
    cudaEvent_t ev[2] = {nullptr, nullptr};
    cudaStream_t st = (cudaStream_t)stream;
    rc = PYJAC_OK;
    if (cudaMalloc(&d_ent, ent.size() * 4) != cudaSuccess || cudaMalloc(&d_hdr, hdr.size() * 4) != cudaSuccess ||
        cudaMalloc(&d_pos, cpos.size() * 2) != cudaSuccess)
        rc = PYJAC_ENOMEM;
    else if (cudaMemcpy(d_ent, ent.data(), ent.size() * 4, cudaMemcpyHostToDevice) != cudaSuccess ||
             cudaMemcpy(d_hdr, hdr.data(), hdr.size() * 4, cudaMemcpyHostToDevice) != cudaSuccess ||
             cudaMemcpy(d_pos, cpos.data(), cpos.size() * 2, cudaMemcpyHostToDevice) != cudaSuccess ||
             cudaFuncSetAttribute(k, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem) != cudaSuccess ||
             cudaEventCreate(&ev[0]) != cudaSuccess || cudaEventCreate(&ev[1]) != cudaSuccess)
        rc = PYJAC_ECUDA;
    if (rc == PYJAC_OK) {
        const long long batches = (n_states + S - 1) / S;
        const int grid = (int)std::min<long long>(batches, (long long)n_sm * ctas_per_sm);
        float best = 1e30f, sum = 0.f;
        for (int it = 0; it < 2 + reps && rc == PYJAC_OK; ++it) {           // two warm-up launches
            cudaEventRecord(ev[0], st);
            k<<<grid, threads, smem, st>>>(d_ent, d_hdr, d_pos, (int)hdr.size(), n_e, ld, hp.eAlpha, hp.eGamma, n_buf,
                                           (long long)n_states, out);
            cudaEventRecord(ev[1], st);
            float ms = 0.f;
            if (cudaGetLastError() != cudaSuccess || cudaEventSynchronize(ev[1]) != cudaSuccess ||
                cudaEventElapsedTime(&ms, ev[0], ev[1]) != cudaSuccess)
                rc = PYJAC_ECUDA;
            else if (it >= 2) { best = std::min(best, ms); sum += ms; }
        }
        *ms_best = best;
        *ms_mean = sum / (float)reps;
        stats[7] = grid;
    }
    if (ev[0]) cudaEventDestroy(ev[0]);
    if (ev[1]) cudaEventDestroy(ev[1]);
    cudaFree(d_ent); cudaFree(d_hdr); cudaFree(d_pos);
    if (rc != PYJAC_OK) cudaGetLastError();
    return rc;
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
