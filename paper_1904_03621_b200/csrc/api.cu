// api.cu -- the C ABI of include/ising.h and the host driver that sequences the kernels.
// No torch types, no exceptions across the boundary, no CPU fallback: without a CUDA device every compute entry
// point returns ISING_ERR_CUDA.
#include <cmath>
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <string>
#include <vector>

#include "common.cuh"
#include "../../include/ising.h"

namespace ising {
namespace {

thread_local std::string t_last_error;
thread_local ising_stats t_stats;
thread_local bool t_have_stats = false;

// Per-host-thread, per-device scratch. Calls of one thread are sequential (each call synchronises its stream
// before returning), so the workspace can be reused; different threads own different workspaces.
struct Workspace {
    int device = -1;
    Entry* pool = nullptr;          // POOL_CAP entries
    Tables* tab = nullptr;
    Ctrl* ctrl = nullptr;
    Ctrl* h_ctrl = nullptr;         // pinned
    double* J2 = nullptr;           // 64*64 converted / staged couplings
    double* h2 = nullptr;           // 64
    unsigned long long* out_q = nullptr;   // ISING_S_MAX
    double* out_e = nullptr;               // ISING_S_MAX
    cudaEvent_t ev[4] = {nullptr, nullptr, nullptr, nullptr};
    void release()
    {
        if (device < 0) return;
        cudaFree(pool); cudaFree(tab); cudaFree(ctrl); cudaFree(J2); cudaFree(h2); cudaFree(out_q); cudaFree(out_e);
        if (h_ctrl) cudaFreeHost(h_ctrl);
        for (auto& e : ev) if (e) cudaEventDestroy(e);
        *this = Workspace();
    }
};
thread_local Workspace t_ws;

#define CUDA_TRY(expr)                                                                              \
    do {                                                                                            \
        cudaError_t err__ = (expr);                                                                 \
        if (err__ != cudaSuccess) {                                                                 \
            t_last_error = std::string(#expr) + ": " + cudaGetErrorString(err__);                   \
            return ISING_ERR_CUDA;                                                                  \
        }                                                                                           \
    } while (0)

int ensure_workspace()
{
    int dev = -1;
    CUDA_TRY(cudaGetDevice(&dev));
    if (t_ws.device == dev) return ISING_OK;
    t_ws.release();
    CUDA_TRY(cudaMalloc(&t_ws.pool, sizeof(Entry) * (size_t)POOL_CAP));
    CUDA_TRY(cudaMalloc(&t_ws.tab, sizeof(Tables)));
    CUDA_TRY(cudaMalloc(&t_ws.ctrl, sizeof(Ctrl)));
    CUDA_TRY(cudaMallocHost(&t_ws.h_ctrl, sizeof(Ctrl)));
    CUDA_TRY(cudaMalloc(&t_ws.J2, sizeof(double) * 64 * 64));
    CUDA_TRY(cudaMalloc(&t_ws.h2, sizeof(double) * 64));
    CUDA_TRY(cudaMalloc(&t_ws.out_q, sizeof(unsigned long long) * ISING_S_MAX));
    CUDA_TRY(cudaMalloc(&t_ws.out_e, sizeof(double) * ISING_S_MAX));
    for (auto& e : t_ws.ev) CUDA_TRY(cudaEventCreate(&e));
    t_ws.device = dev;
    return ISING_OK;
}

int floor_log2(unsigned long long x)
{
    int r = -1;
    while (x) { x >>= 1; ++r; }
    return r;
}

int env_int(const char* name, int dflt, int lo, int hi)
{
    const char* s = getenv(name);
    if (!s || !*s) return dflt;
    int v = atoi(s);
    return v < lo ? lo : (v > hi ? hi : v);
}

__global__ void reset_count_kernel(Ctrl* ctrl) { ctrl->count = ctrl->kept; }

struct Piece {
    unsigned long long base;
    unsigned nthreads;
    int Lw;
    bool direct;                    // the priming piece: one thread per state (direct_kernel)
};

// mode 0: (J, h) is an Ising instance, energies by eq. (1). mode 1: (Jorig, horig) = QUBO (a, b); (J, h) its Ising image.
int run_lowest(const double* J, const double* h, const double* Jorig, const double* horig, int mode, double extra_eps_rel,
               int N, int S, unsigned long long q_begin, unsigned long long q_end,
               unsigned long long* states_out, double* energies_out, cudaStream_t st)
{
    Workspace& ws = t_ws;
    ising_stats stats;
    memset(&stats, 0, sizeof(stats));
    const int lw_run = env_int("ISING_LW", LW_MAX, 0, LW_MAX);
    const int chunk_log2 = env_int("ISING_CHUNK_LOG2", 42, MIN_CHUNK_BITS, 44);
    const int growth = env_int("ISING_GROWTH", 3, 1, 1 << 20);   // a launch is at most growth x what has been processed
    const int variant = env_int("ISING_KERNEL", 16, 16, 32) == 32 ? 32 : 16;   // 16: packed screen, 32: int32 kernel

    CUDA_TRY(cudaEventRecord(ws.ev[0], st));
    launch_stage(J, h, N, ws.tab, ws.ctrl, st, extra_eps_rel);
    stats.kernel_launches += 2;
    CUDA_TRY(cudaMemcpyAsync(ws.h_ctrl, ws.ctrl, sizeof(Ctrl), cudaMemcpyDeviceToHost, st));
    CUDA_TRY(cudaStreamSynchronize(st));
    if (ws.h_ctrl->status != ISING_OK) {
        t_last_error = std::string("instance rejected: ") + ising_strerror(ws.h_ctrl->status);
        return ws.h_ctrl->status;
    }
    stats.grid_exponent = ws.h_ctrl->p;
    stats.exact = ws.h_ctrl->exact;
    stats.epsilon = ws.h_ctrl->epsilon;
    stats.inner_bits = LOWBITS;
    stats.kernel_variant = variant;
    stats.screen_shift = variant == 16 ? ws.h_ctrl->shift16 : -1;
    stats.passes = 1;

    double enum_ms = 0.0;
    unsigned kept = 0;
    if (N <= N_DIRECT_MAX) {
        launch_direct(ws.tab, ws.ctrl, ws.pool, N, 0, 1u << N, 0, st);
        stats.kernel_launches += 1;
        stats.enum_launches += 1;
        stats.configs = 1ull << N;
        stats.candidates = 1ull << N;
        stats.kernel_launches += launch_select(ws.pool, ws.ctrl, 1u << N, S, st);
    } else {
        unsigned long long cur = q_begin, processed = 0;
        std::vector<Piece> stack;
        bool tau_finite = false;
        while (cur < q_end || !stack.empty()) {
            Piece pc;
            if (!stack.empty()) {
                pc = stack.back();
                stack.pop_back();
            } else {
                const unsigned long long remaining = q_end - cur;
                unsigned long long target = 1ull << MIN_CHUNK_BITS;
                if (processed > 0) {
                    target = (unsigned long long)growth * processed;
                    if (target > (1ull << chunk_log2)) target = 1ull << chunk_log2;
                    if (!tau_finite && target > (1ull << 16)) target = 1ull << 16;   // everything passes: keep it small
                }
                const unsigned long long sz = target < remaining ? target : remaining;
                int Lw = floor_log2(sz) - 27;
                Lw = Lw < 0 ? 0 : (Lw > lw_run ? lw_run : Lw);
                while (Lw > 0 && (cur & ((1ull << (LOWBITS + Lw)) - 1))) --Lw;
                unsigned long long nt = (sz >> (LOWBITS + Lw)) / 32 * 32;
                if (nt < 32 || nt > 0x7fffffe0ull) {
                    t_last_error = "internal: bad launch plan";
                    return ISING_ERR_INTERNAL;
                }
                pc.base = cur;
                pc.nthreads = (unsigned)nt;
                pc.Lw = Lw;
                pc.direct = (processed == 0);          // a2': the first 2^15 states, tau = +inf
                cur += nt << (LOWBITS + Lw);
            }
            CUDA_TRY(cudaEventRecord(ws.ev[2], st));
            if (pc.direct) launch_direct(ws.tab, ws.ctrl, ws.pool, N, pc.base, pc.nthreads << (LOWBITS + pc.Lw), 0, st);
            else if (variant == 16) launch_enumerate16(ws.tab, ws.ctrl, ws.pool, N, pc.Lw, pc.base, pc.nthreads,
                                                       processed < (1ull << 30), st);
            else launch_enumerate(ws.tab, ws.ctrl, ws.pool, N, pc.Lw, pc.base, pc.nthreads, st);
            CUDA_TRY(cudaEventRecord(ws.ev[3], st));
            stats.kernel_launches += 1;
            stats.enum_launches += 1;
            CUDA_TRY(cudaMemcpyAsync(ws.h_ctrl, ws.ctrl, sizeof(Ctrl), cudaMemcpyDeviceToHost, st));
            CUDA_TRY(cudaStreamSynchronize(st));
            float ms = 0.f;
            CUDA_TRY(cudaEventElapsedTime(&ms, ws.ev[2], ws.ev[3]));
            enum_ms += ms;
            const unsigned count = ws.h_ctrl->count;
            kept = ws.h_ctrl->kept;
            const unsigned long long pc_size = (unsigned long long)pc.nthreads << (LOWBITS + pc.Lw);
            if (count > POOL_CAP) {
                // pool overflow: drop this piece's candidates and run it again in two halves
                reset_count_kernel<<<1, 1, 0, st>>>(ws.ctrl);
                stats.kernel_launches += 1;
                stats.split_retries += 1;
                Piece a = pc, b = pc;
                a.direct = b.direct = false;
                if (pc.nthreads >= 64) {
                    a.nthreads = pc.nthreads / 64 * 32;
                    b.nthreads = pc.nthreads - a.nthreads;
                    b.base = pc.base + ((unsigned long long)a.nthreads << (LOWBITS + pc.Lw));
                } else if (pc.Lw > 0) {
                    a.Lw = b.Lw = pc.Lw - 1;
                    b.base = pc.base + (32ull << (LOWBITS + a.Lw));
                } else {
                    t_last_error = "internal: candidate pool overflow on a minimal launch";
                    return ISING_ERR_INTERNAL;
                }
                stack.push_back(b);
                stack.push_back(a);
                continue;
            }
            processed += pc_size;
            stats.configs += pc_size;
            stats.candidates += count - kept;
            if (count > kept) {
                stats.kernel_launches += launch_select(ws.pool, ws.ctrl, count, S, st);
                if (count >= (unsigned)S) tau_finite = true;
            }
        }
    }
    CUDA_TRY(cudaMemcpyAsync(ws.h_ctrl, ws.ctrl, sizeof(Ctrl), cudaMemcpyDeviceToHost, st));
    CUDA_TRY(cudaStreamSynchronize(st));
    if (ws.h_ctrl->band_overflow) {
        t_last_error = "guard band holds more than KEEP_CAP states; the S-th level cannot be certified";
        return ISING_ERR_BAND;
    }
    kept = ws.h_ctrl->kept;
    if (kept < (unsigned)S) {
        t_last_error = "internal: fewer states kept than requested";
        return ISING_ERR_INTERNAL;
    }
    stats.keep = (int)kept;
    stats.kernel_launches += launch_final(mode ? Jorig : J, mode ? horig : h, N, mode, ws.pool, kept, S,
                                          states_out, energies_out, st);
    CUDA_TRY(cudaEventRecord(ws.ev[1], st));
    CUDA_TRY(cudaStreamSynchronize(st));
    CUDA_TRY(cudaGetLastError());
    float total_ms = 0.f;
    CUDA_TRY(cudaEventElapsedTime(&total_ms, ws.ev[0], ws.ev[1]));
    stats.enum_ms = enum_ms;
    stats.total_ms = total_ms;
    t_stats = stats;
    t_have_stats = true;
    return ISING_OK;
}

int check_args(const void* J, const void* h, int N, int S, unsigned long long q_begin, unsigned long long q_end,
               const void* so, const void* eo)
{
    if (!J || !h || !so || !eo) { t_last_error = "null pointer argument"; return ISING_ERR_NULL; }
    if (N < 1 || N > ISING_N_MAX) { t_last_error = "N out of range"; return ISING_ERR_BAD_N; }
    const unsigned long long total = 1ull << N;
    const unsigned long long unit = 1ull << (N < 20 ? N : 20);
    if (q_begin >= q_end || q_end > total || (q_begin % unit) || (q_end % unit)) {
        t_last_error = "bad state range";
        return ISING_ERR_BAD_RANGE;
    }
    if (S < 1 || S > ISING_S_MAX || (unsigned long long)S > q_end - q_begin) {
        t_last_error = "S out of range";
        return ISING_ERR_BAD_S;
    }
    return ISING_OK;
}

}  // namespace
}  // namespace ising

using namespace ising;

extern "C" {

int ising_lowest_range(const double* J_dev, const double* h_dev, int N, int S, uint64_t q_begin, uint64_t q_end,
                       uint64_t* states_out_dev, double* energies_out_dev, void* stream)
{
    t_last_error.clear();
    int rc = check_args(J_dev, h_dev, N, S, q_begin, q_end, states_out_dev, energies_out_dev);
    if (rc != ISING_OK) return rc;
    rc = ensure_workspace();
    if (rc != ISING_OK) return rc;
    return run_lowest(J_dev, h_dev, nullptr, nullptr, 0, 0.0, N, S, q_begin, q_end,
                      (unsigned long long*)states_out_dev, energies_out_dev, (cudaStream_t)stream);
}

int ising_lowest(const double* J_dev, const double* h_dev, int N, int S, uint64_t* states_out_dev,
                 double* energies_out_dev, void* stream)
{
    if (N < 1 || N > ISING_N_MAX) { t_last_error = "N out of range"; return ISING_ERR_BAD_N; }
    return ising_lowest_range(J_dev, h_dev, N, S, 0, 1ull << N, states_out_dev, energies_out_dev, stream);
}

int ising_lowest_host(const double* J_host, const double* h_host, int N, int S, uint64_t q_begin, uint64_t q_end,
                      uint64_t* states_out_host, double* energies_out_host, void* stream)
{
    t_last_error.clear();
    int rc = check_args(J_host, h_host, N, S, q_begin, q_end, states_out_host, energies_out_host);
    if (rc != ISING_OK) return rc;
    rc = ensure_workspace();
    if (rc != ISING_OK) return rc;
    cudaStream_t st = (cudaStream_t)stream;
    Workspace& ws = t_ws;
    CUDA_TRY(cudaMemcpyAsync(ws.J2, J_host, sizeof(double) * N * N, cudaMemcpyHostToDevice, st));
    CUDA_TRY(cudaMemcpyAsync(ws.h2, h_host, sizeof(double) * N, cudaMemcpyHostToDevice, st));
    rc = run_lowest(ws.J2, ws.h2, nullptr, nullptr, 0, 0.0, N, S, q_begin, q_end, ws.out_q, ws.out_e, st);
    if (rc != ISING_OK) return rc;
    CUDA_TRY(cudaMemcpyAsync(states_out_host, ws.out_q, sizeof(uint64_t) * S, cudaMemcpyDeviceToHost, st));
    CUDA_TRY(cudaMemcpyAsync(energies_out_host, ws.out_e, sizeof(double) * S, cudaMemcpyDeviceToHost, st));
    CUDA_TRY(cudaStreamSynchronize(st));
    return ISING_OK;
}

int ising_dos(const double* J_dev, const double* h_dev, int N, int nbins, uint64_t* hist_out_dev,
              double* e_lo_out_host, double* bin_width_out_host, void* stream)
{
    t_last_error.clear();
    if (!J_dev || !h_dev || !hist_out_dev || !e_lo_out_host || !bin_width_out_host) {
        t_last_error = "null pointer argument";
        return ISING_ERR_NULL;
    }
    if (N < 1 || N > ISING_N_MAX) { t_last_error = "N out of range"; return ISING_ERR_BAD_N; }
    if (nbins < 2 || nbins > 4096) { t_last_error = "nbins must be in [2, 4096]"; return ISING_ERR_BAD_S; }
    int rc = ensure_workspace();
    if (rc != ISING_OK) return rc;
    cudaStream_t st = (cudaStream_t)stream;
    Workspace& ws = t_ws;
    ising_stats stats;
    memset(&stats, 0, sizeof(stats));
    CUDA_TRY(cudaEventRecord(ws.ev[0], st));
    launch_stage(J_dev, h_dev, N, ws.tab, ws.ctrl, st, 0.0);
    stats.kernel_launches += 2;
    CUDA_TRY(cudaMemcpyAsync(ws.h_ctrl, ws.ctrl, sizeof(Ctrl), cudaMemcpyDeviceToHost, st));
    CUDA_TRY(cudaStreamSynchronize(st));
    if (ws.h_ctrl->status != ISING_OK) {
        t_last_error = std::string("instance rejected: ") + ising_strerror(ws.h_ctrl->status);
        return ws.h_ctrl->status;
    }
    const int p = ws.h_ctrl->p;
    // every grid energy lies in [-Wq, Wq], Wq = sum of the rounded |weights| <= W 2^p + (number of weights)
    const long long Wq = (long long)ceil(ldexp(ws.h_ctrl->W, p)) + (long long)N * (N - 1) / 2 + N + 1;
    const long long e_lo = -Wq;
    int bshift = 0;
    while (((2 * Wq) >> bshift) + 1 > (long long)nbins) ++bshift;
    CUDA_TRY(cudaMemsetAsync(hist_out_dev, 0, sizeof(uint64_t) * (size_t)nbins, st));
    if (N <= N_DIRECT_MAX) {
        launch_dos_direct(ws.tab, N, (int)e_lo, bshift, (unsigned long long*)hist_out_dev, st);
        stats.kernel_launches += 1;
        stats.enum_launches += 1;
    } else {
        int Lw = N - LOWBITS - 12;
        Lw = Lw < 0 ? 0 : (Lw > LW_MAX ? LW_MAX : Lw);
        const unsigned long long total_threads = 1ull << (N - LOWBITS - Lw);       // >= 32 because N >= 15
        const unsigned long long per_launch = 1ull << 22;
        for (unsigned long long t0 = 0; t0 < total_threads; t0 += per_launch) {
            const unsigned nt = (unsigned)((total_threads - t0) < per_launch ? (total_threads - t0) : per_launch);
            launch_dos(ws.tab, N, Lw, t0 << (LOWBITS + Lw), nt, (int)e_lo, bshift, nbins,
                       (unsigned long long*)hist_out_dev, st);
            stats.kernel_launches += 1;
            stats.enum_launches += 1;
        }
    }
    CUDA_TRY(cudaEventRecord(ws.ev[1], st));
    CUDA_TRY(cudaStreamSynchronize(st));
    CUDA_TRY(cudaGetLastError());
    float total_ms = 0.f;
    CUDA_TRY(cudaEventElapsedTime(&total_ms, ws.ev[0], ws.ev[1]));
    *e_lo_out_host = ldexp((double)e_lo, -p);
    *bin_width_out_host = ldexp(1.0, bshift - p);
    stats.configs = 1ull << N;
    stats.grid_exponent = p;
    stats.exact = ws.h_ctrl->exact;
    stats.epsilon = ws.h_ctrl->epsilon;
    stats.total_ms = total_ms;
    stats.enum_ms = total_ms;
    stats.passes = 1;
    stats.kernel_variant = 2;
    stats.screen_shift = -1;
    stats.inner_bits = LOWBITS;
    t_stats = stats;
    t_have_stats = true;
    return ISING_OK;
}

int ising_lowest_alg1(const double* J_dev, const double* h_dev, int N, int S, uint64_t q_begin, uint64_t q_end,
                      int chunk_log2, uint64_t* states_out_dev, double* energies_out_dev, void* stream)
{
    t_last_error.clear();
    int rc = check_args(J_dev, h_dev, N, S, q_begin, q_end, states_out_dev, energies_out_dev);
    if (rc != ISING_OK) return rc;
    if (chunk_log2 < 10 || chunk_log2 > 20) { t_last_error = "chunk_log2 must be in [10, 20]"; return ISING_ERR_BAD_RANGE; }
    rc = ensure_workspace();
    if (rc != ISING_OK) return rc;
    cudaStream_t st = (cudaStream_t)stream;
    Workspace& ws = t_ws;
    ising_stats stats;
    memset(&stats, 0, sizeof(stats));
    CUDA_TRY(cudaEventRecord(ws.ev[0], st));
    launch_stage(J_dev, h_dev, N, ws.tab, ws.ctrl, st, 0.0);          // validation only (same error codes)
    stats.kernel_launches += 2;
    CUDA_TRY(cudaMemcpyAsync(ws.h_ctrl, ws.ctrl, sizeof(Ctrl), cudaMemcpyDeviceToHost, st));
    CUDA_TRY(cudaStreamSynchronize(st));
    if (ws.h_ctrl->status != ISING_OK && ws.h_ctrl->status != ISING_ERR_RANGE_W) {
        t_last_error = std::string("instance rejected: ") + ising_strerror(ws.h_ctrl->status);
        return ws.h_ctrl->status;
    }
    unsigned kept = 0;
    const unsigned long long chunk = 1ull << chunk_log2;
    for (unsigned long long cur = q_begin; cur < q_end; cur += chunk) {
        const unsigned cnt = (unsigned)((q_end - cur) < chunk ? (q_end - cur) : chunk);
        stats.kernel_launches += launch_alg1_chunk(J_dev, h_dev, N, cur, cnt, ws.pool, kept, st);
        stats.enum_launches += 1;
        stats.configs += cnt;
        stats.candidates += cnt;
        kept = kept + cnt < (unsigned)S ? kept + cnt : (unsigned)S;
    }
    stats.kernel_launches += launch_emit(ws.pool, S, (unsigned long long*)states_out_dev, energies_out_dev, st);
    CUDA_TRY(cudaEventRecord(ws.ev[1], st));
    CUDA_TRY(cudaStreamSynchronize(st));
    CUDA_TRY(cudaGetLastError());
    float total_ms = 0.f;
    CUDA_TRY(cudaEventElapsedTime(&total_ms, ws.ev[0], ws.ev[1]));
    stats.total_ms = total_ms;
    stats.enum_ms = total_ms;
    stats.exact = 1;
    stats.keep = S;
    stats.passes = 1;
    stats.kernel_variant = 1;
    stats.screen_shift = -1;
    t_stats = stats;
    t_have_stats = true;
    return ISING_OK;
}

int ising_lowest_h0(const double* J_dev, int N, int S, uint64_t* states_out_dev, double* energies_out_dev, void* stream)
{
    t_last_error.clear();
    if (N < 1 || N > ISING_N_MAX) { t_last_error = "N out of range"; return ISING_ERR_BAD_N; }
    int rc = check_args(J_dev, J_dev, N, S, 0, 1ull << N, states_out_dev, energies_out_dev);
    if (rc != ISING_OK) return rc;
    rc = ensure_workspace();
    if (rc != ISING_OK) return rc;
    cudaStream_t st = (cudaStream_t)stream;
    Workspace& ws = t_ws;
    CUDA_TRY(cudaMemsetAsync(ws.h2, 0, sizeof(double) * 64, st));
    if (N <= 20)      // too small for a half-space range (ranges are multiples of 2^min(N,20)): plain call
        return run_lowest(J_dev, ws.h2, nullptr, nullptr, 0, 0.0, N, S, 0, 1ull << N,
                          (unsigned long long*)states_out_dev, energies_out_dev, st);
    const unsigned long long half = 1ull << (N - 1);
    const int S_half = (unsigned long long)S < half ? S : (int)half;
    rc = run_lowest(J_dev, ws.h2, nullptr, nullptr, 0, 0.0, N, S_half, 0, half, ws.out_q, ws.out_e, st);
    if (rc != ISING_OK) return rc;
    t_stats.kernel_launches += launch_expand_complements(ws.out_q, ws.out_e, S_half, N, S, ws.pool,
                                                         (unsigned long long*)states_out_dev, energies_out_dev, st);
    CUDA_TRY(cudaStreamSynchronize(st));
    CUDA_TRY(cudaGetLastError());
    return ISING_OK;
}

int qubo_lowest(const double* a_dev, const double* b_dev, int N, int S, uint64_t* states_out_dev,
                double* energies_out_dev, void* stream)
{
    t_last_error.clear();
    if (N < 1 || N > ISING_N_MAX) { t_last_error = "N out of range"; return ISING_ERR_BAD_N; }
    int rc = check_args(a_dev, b_dev, N, S, 0, 1ull << N, states_out_dev, energies_out_dev);
    if (rc != ISING_OK) return rc;
    rc = ensure_workspace();
    if (rc != ISING_OK) return rc;
    cudaStream_t st = (cudaStream_t)stream;
    Workspace& ws = t_ws;
    launch_qubo_to_ising(a_dev, b_dev, N, ws.J2, ws.h2, st);
    // h = b/2 + sum a/4 is rounded in fp64: widen the band by a relative 2^-40 of W (far above N ulps)
    return run_lowest(ws.J2, ws.h2, a_dev, b_dev, 1, 9.1e-13, N, S, 0, 1ull << N,
                      (unsigned long long*)states_out_dev, energies_out_dev, st);
}

int ising_merge_lists(const uint64_t* states_in_dev, const double* energies_in_dev, int64_t n, int S,
                      uint64_t* states_out_dev, double* energies_out_dev, void* stream)
{
    t_last_error.clear();
    if (!states_in_dev || !energies_in_dev || !states_out_dev || !energies_out_dev) {
        t_last_error = "null pointer argument";
        return ISING_ERR_NULL;
    }
    if (n < 1 || n > (int64_t)POOL_CAP || S < 1 || S > n) { t_last_error = "bad n or S"; return ISING_ERR_BAD_S; }
    int rc = ensure_workspace();
    if (rc != ISING_OK) return rc;
    cudaStream_t st = (cudaStream_t)stream;
    launch_merge_lists((const unsigned long long*)states_in_dev, energies_in_dev, n, S, t_ws.pool,
                       (unsigned long long*)states_out_dev, energies_out_dev, st);
    CUDA_TRY(cudaStreamSynchronize(st));
    CUDA_TRY(cudaGetLastError());
    return ISING_OK;
}

int ising_energies(const double* J_dev, const double* h_dev, int N, const uint64_t* states_dev, int64_t n,
                   double* energies_out_dev, void* stream)
{
    t_last_error.clear();
    if (!J_dev || !h_dev || !states_dev || !energies_out_dev) { t_last_error = "null pointer argument"; return ISING_ERR_NULL; }
    if (N < 1 || N > ISING_N_MAX) { t_last_error = "N out of range"; return ISING_ERR_BAD_N; }
    if (n < 0) { t_last_error = "negative count"; return ISING_ERR_BAD_S; }
    cudaStream_t st = (cudaStream_t)stream;
    launch_energies(J_dev, h_dev, N, 0, (const unsigned long long*)states_dev, n, energies_out_dev, st);
    CUDA_TRY(cudaStreamSynchronize(st));
    CUDA_TRY(cudaGetLastError());
    return ISING_OK;
}

int ising_get_last_stats(ising_stats* out_host)
{
    if (!out_host) return ISING_ERR_NULL;
    if (!t_have_stats) return ISING_ERR_INTERNAL;
    *out_host = t_stats;
    return ISING_OK;
}

const char* ising_strerror(int status)
{
    switch (status) {
        case ISING_OK: return "ok";
        case ISING_ERR_NULL: return "a required pointer is NULL";
        case ISING_ERR_BAD_N: return "N out of range";
        case ISING_ERR_BAD_S: return "S out of range";
        case ISING_ERR_NONFINITE: return "NaN or Inf in J or h";
        case ISING_ERR_ASYMMETRIC: return "J is not symmetric";
        case ISING_ERR_DIAGONAL: return "J has a non-zero diagonal";
        case ISING_ERR_BAD_RANGE: return "bad state range";
        case ISING_ERR_CUDA: return "CUDA runtime error";
        case ISING_ERR_BAND: return "guard band could not certify the result";
        case ISING_ERR_INTERNAL: return "internal error";
        case ISING_ERR_RANGE_W: return "weights cannot be put on a 2^-p grid";
        default: return "unknown status";
    }
}

const char* ising_last_error(void) { return t_last_error.c_str(); }

int ising_version(void) { return 100; }

int ising_fma_peak(double ms_target, double* fma_per_s_out_host, void* stream)
{
    if (!fma_per_s_out_host) return ISING_ERR_NULL;
    double r = run_fma_peak(ms_target, (cudaStream_t)stream, 0);
    if (r < 0.0) { t_last_error = "FFMA microbenchmark failed"; return ISING_ERR_CUDA; }
    *fma_per_s_out_host = r;
    return ISING_OK;
}

int ising_addmin_peak(double ms_target, double* addmin_per_s_out_host, void* stream)
{
    if (!addmin_per_s_out_host) return ISING_ERR_NULL;
    double r = run_fma_peak(ms_target, (cudaStream_t)stream, 1);
    if (r < 0.0) { t_last_error = "VIADDMNMX microbenchmark failed"; return ISING_ERR_CUDA; }
    *addmin_per_s_out_host = r;
    return ISING_OK;
}

int ising_addmin16x2_peak(double ms_target, double* inst_per_s_out_host, void* stream)
{
    if (!inst_per_s_out_host) return ISING_ERR_NULL;
    double r = run_fma_peak(ms_target, (cudaStream_t)stream, 2);
    if (r < 0.0) { t_last_error = "VIADDMNMX.U16x2 microbenchmark failed"; return ISING_ERR_CUDA; }
    *inst_per_s_out_host = r;
    return ISING_OK;
}

void ising_release_workspace(void) { t_ws.release(); }

}  // extern "C"
