// api.cu -- the C ABI of include/ising.h and the host driver that sequences the kernels.
// No torch types, no exceptions across the boundary, no CPU fallback: without a CUDA device every compute entry
// point returns ISING_ERR_CUDA.
#include <cmath>
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <string>
#include <vector>
#include <climits>

#include "common.cuh"
#include "../../include/ising.h"

namespace ising {
namespace {

thread_local std::string t_last_error;
thread_local ising_stats t_stats;
thread_local bool t_have_stats = false;

// Per-host-thread, per-device scratch. Calls of one thread are sequential (each call synchronises its stream
// before returning), so the workspace can be reused; different threads own different workspaces. Freed when the
// thread exits (or by ising_release_workspace); a partly failed allocation is freed before the error is returned.
struct Workspace {
    int device = -1;
    Entry* pool = nullptr;          // POOL_CAP entries: candidates
    Entry* pool2 = nullptr;         // POOL_CAP entries: compacted candidates / band-pass scratch
    unsigned* hist = nullptr;       // HIST_WORDS counters: candidate histogram (walk.cuh)
    Tables* tab = nullptr;
    ZTables* zt = nullptr;          // tables of the tensor-core screen
    Ctrl* ctrl = nullptr;
    Ctrl* h_ctrl = nullptr;         // pinned
    double* J2 = nullptr;           // 64*64 converted / staged couplings
    double* h2 = nullptr;           // 64
    unsigned long long* out_q = nullptr;   // ISING_S_MAX
    double* out_e = nullptr;               // ISING_S_MAX
    cudaEvent_t ev[4] = {nullptr, nullptr, nullptr, nullptr};
    void release()
    {
        cudaFree(pool); cudaFree(pool2); cudaFree(hist); cudaFree(tab); cudaFree(zt); cudaFree(ctrl); cudaFree(J2); cudaFree(h2);
        cudaFree(out_q); cudaFree(out_e);
        if (h_ctrl) cudaFreeHost(h_ctrl);
        for (auto& e : ev) if (e) cudaEventDestroy(e);
        pool = pool2 = nullptr; hist = nullptr; tab = nullptr; zt = nullptr; ctrl = h_ctrl = nullptr; J2 = h2 = nullptr;
        out_q = nullptr; out_e = nullptr;
        for (auto& e : ev) e = nullptr;
        device = -1;
    }
    ~Workspace() { if (device >= 0) release(); }
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

// after a kernel launch: a failed launch is reported at once, under the kernel's name
#define LAUNCH_CHECK(name)                                                                          \
    do {                                                                                            \
        cudaError_t err__ = cudaGetLastError();                                                     \
        if (err__ != cudaSuccess) {                                                                 \
            t_last_error = std::string("launch of ") + (name) + ": " + cudaGetErrorString(err__);   \
            return ISING_ERR_CUDA;                                                                  \
        }                                                                                           \
    } while (0)

int allocate_workspace(Workspace& ws, int dev)
{
    CUDA_TRY(cudaMalloc(&ws.pool, sizeof(Entry) * (size_t)POOL_CAP));
    CUDA_TRY(cudaMalloc(&ws.pool2, sizeof(Entry) * (size_t)POOL_CAP));
    CUDA_TRY(cudaMalloc(&ws.hist, sizeof(unsigned) * (size_t)HIST_WORDS));
    CUDA_TRY(cudaMalloc(&ws.tab, sizeof(Tables)));
    CUDA_TRY(cudaMalloc(&ws.zt, sizeof(ZTables)));
    CUDA_TRY(cudaMalloc(&ws.ctrl, sizeof(Ctrl)));
    CUDA_TRY(cudaMallocHost(&ws.h_ctrl, sizeof(Ctrl)));
    CUDA_TRY(cudaMalloc(&ws.J2, sizeof(double) * 64 * 64));
    CUDA_TRY(cudaMalloc(&ws.h2, sizeof(double) * 64));
    CUDA_TRY(cudaMalloc(&ws.out_q, sizeof(unsigned long long) * ISING_S_MAX));
    CUDA_TRY(cudaMalloc(&ws.out_e, sizeof(double) * ISING_S_MAX));
    for (auto& e : ws.ev) CUDA_TRY(cudaEventCreate(&e));
    (void)dev;
    set_select_attributes();                       // per-device function attributes (dynamic shared memory)
    set_zscreen_attributes();
    CUDA_TRY(cudaGetLastError());
    return ISING_OK;
}

int ensure_workspace()
{
    int dev = -1;
    CUDA_TRY(cudaGetDevice(&dev));
    if (t_ws.device == dev) return ISING_OK;
    t_ws.release();
    const int rc = allocate_workspace(t_ws, dev);
    if (rc != ISING_OK) { t_ws.release(); return rc; }
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

// host-sequenced path: between launches
__global__ void reset_queue_kernel(Ctrl* ctrl, int drop_new)
{
    ctrl->next_unit = 0ull;                 // done_configs keeps counting: Segment::need_done is relative to q_begin
    if (drop_new) { ctrl->count = ctrl->kept; ctrl->pool_overflow = 0u; }
}
// restart of a whole run (after a void single-pass attempt) or start of the band pass
__global__ void restart_kernel(Ctrl* ctrl, unsigned long long tau)
{
    ctrl->next_unit = 0ull;
    ctrl->done_configs = 0ull;
    ctrl->count = 0u;
    ctrl->kept = 0u;
    ctrl->pool_overflow = 0u;
    ctrl->band_overflow = 0u;
    ctrl->count2 = 0u;
    ctrl->final_state = 0u;
    ctrl->tau = tau;
}
// band pass: the sure states (grid energy below the band; a sorted prefix of pool) move to pool2, keyed by fp64 energy
__global__ void count_sure_kernel(const Entry* __restrict__ pool, Ctrl* __restrict__ ctrl, unsigned kept, int band)
{
    if (threadIdx.x != 0 || blockIdx.x != 0) return;
    const unsigned long long klim = key_from_i32(ctrl->eS - band);       // sure: key < klim
    unsigned lo = 0, hi = kept;
    while (lo < hi) {
        const unsigned mid = (lo + hi) >> 1;
        if (pool[mid].key < klim) lo = mid + 1; else hi = mid;
    }
    ctrl->n_sure = lo;
}
__global__ void copy_entries_kernel(const Entry* __restrict__ src, Entry* __restrict__ dst, unsigned n)
{
    const unsigned i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i < n) dst[i] = src[i];
}

// One call's invariants, shared by the three host paths below.
struct Run {
    Workspace* ws;
    ising_stats* stats;
    const double *J, *h, *Jorig, *horig;
    int mode, N, S, variant, lw_max, chunk_log2, growth, qshift, z_min_log2, z_ramp_log2, z_force;
    unsigned keep_cap;
    unsigned long long q_begin, q_end;
    cudaStream_t st;
    double enum_ms;
    double z_ms;                    // of which in launches of the tensor-core screen
    unsigned long long z_configs;   // configurations those launches covered
    bool done;                      // the single pass wrote the outputs and recorded the end event
};

void plan_header(const Run& r, Plan& plan, int use_hist, int loE)
{
    memset(&plan, 0, sizeof(plan));
    plan.q_begin = r.q_begin;
    plan.q_end = r.q_end;
    plan.N = r.N;
    plan.S = r.S;
    plan.use_hist = use_hist;
    const int rf = r.S / 8;
    plan.refresh = rf < 64 ? 64 : rf;
    plan.qshift = r.qshift;
    plan.loE = loE;
    plan.keep_cap = r.keep_cap;
}

// Walk-bit count of a segment of sz configurations at cur: enough units to balance the persistent warps, aligned.
int choose_lw(unsigned long long cur, unsigned long long sz, int lw_max)
{
    // about 2^11 units per segment: a unit costs about two Gray steps to set up (queue, base state, tables), so short
    // units are expensive (measured on cfg2: 2^13 units per segment 0.59 ms, 2^12 0.55 ms, 2^11 0.49 ms per call);
    // the tail of the last segment is tapered instead (run_single_pass)
    int Lw = floor_log2(sz) - MIN_CHUNK_BITS - 11;
    Lw = Lw < 0 ? 0 : (Lw > lw_max ? lw_max : Lw);
    while (Lw > 0 && (cur & ((1ull << (MIN_CHUNK_BITS + Lw)) - 1ull))) --Lw;
    return Lw;
}

int launch_walk(const Run& r, const Plan& plan)
{
    Workspace& ws = *r.ws;
    if (plan.total_units > 0x7fffffffull * WALK_WARPS) { t_last_error = "internal: too many units in one launch"; return ISING_ERR_INTERNAL; }
    if (r.variant != 32) launch_walk16(ws.tab, ws.ctrl, ws.pool, ws.hist, plan, r.st);
    else launch_walk32(ws.tab, ws.ctrl, ws.pool, ws.hist, plan, r.st);
    LAUNCH_CHECK(r.variant != 32 ? "walk_kernel<Inner16>" : "walk_kernel<Inner32>");
    r.stats->kernel_launches += 1;
    r.stats->enum_launches += 1;
    return ISING_OK;
}

// One launch of the tensor-core screen. The grid is one CTA per unit: a count that does not fit the grid's x extent
// (N near 63 in one call, or a small ISING_LW on a huge range) is refused here instead of being truncated.
int launch_z(const Run& r, const Plan& plan)
{
    Workspace& ws = *r.ws;
    if (plan.total_units == 0 || plan.total_units > 0x7fffffffull) {
        t_last_error = "internal: unit count of the tensor-core screen does not fit one launch (split the range)";
        return ISING_ERR_INTERNAL;
    }
    launch_zwalk(ws.tab, ws.zt, ws.ctrl, ws.pool, ws.hist, plan, r.st);
    LAUNCH_CHECK("zwalk_kernel");
    return ISING_OK;
}

int read_ctrl(const Run& r)
{
    CUDA_TRY(cudaMemcpyAsync(r.ws->h_ctrl, r.ws->ctrl, sizeof(Ctrl), cudaMemcpyDeviceToHost, r.st));
    CUDA_TRY(cudaStreamSynchronize(r.st));
    return ISING_OK;
}

// Segments of walked units for the states [cur, to): doubling while `doubling`, then (if `to` is the end of the range)
// a last segment that takes all the rest and tapers its unit size so that the tail stays short.
int plan_walk_segments(const Run& r, Plan& plan, int& ns, unsigned long long& cur, unsigned long long& units,
                       unsigned long long to, unsigned long long need_floor)
{
    auto add_segment = [&](unsigned long long sz, int unit_bits, unsigned long long need) {
        const unsigned long long nu = sz >> unit_bits;
        plan.seg[ns] = Segment{cur, units, nu, need, unit_bits, 0};
        units += nu;
        cur += nu << unit_bits;
        ++ns;
    };
    while (cur < to) {
        const unsigned long long processed = cur - r.q_begin, remaining = to - cur;
        const unsigned long long need = processed / 2 > need_floor ? processed / 2 : need_floor;
        const unsigned long long target = (unsigned long long)r.growth * processed;
        if (ns >= MAX_SEGMENTS - 12) { t_last_error = "internal: bad work plan"; return ISING_ERR_INTERNAL; }
        if (target < remaining && target < (1ull << r.chunk_log2)) {
            const int Lw = choose_lw(cur, target, r.lw_max);
            add_segment(target, MIN_CHUNK_BITS + Lw, need);
            continue;
        }
        // last segment(s): 7/8 of what is left at the full walk length, then 7/8 of the rest with 8x shorter units, ...
        int Lw = choose_lw(cur, remaining, r.lw_max);
        while (cur < to) {
            const unsigned long long left = to - cur;
            while (Lw > 0 && (cur & ((1ull << (MIN_CHUNK_BITS + Lw)) - 1ull))) --Lw;         // alignment of cur
            unsigned long long sz = left;                                                  // Lw = 0: all of it
            if (Lw > 0) sz = (left - (left >> 3)) >> (MIN_CHUNK_BITS + Lw) << (MIN_CHUNK_BITS + Lw);
            if (sz >> (MIN_CHUNK_BITS + Lw)) {
                if (ns >= MAX_SEGMENTS) { t_last_error = "internal: bad work plan"; return ISING_ERR_INTERNAL; }
                add_segment(sz, MIN_CHUNK_BITS + Lw, need);
            }
            Lw = Lw > 3 ? Lw - 3 : 0;
        }
    }
    return ISING_OK;
}

// Segments of tensor-core-screen units (2^(21 + Lw) configurations, one CTA each) for [cur, to), tapered at the end.
// A CTA costs about 20 us before its first step (table copy, tensor-memory allocation, base state) and 3 us per step,
// so units shorter than 2^5 steps are avoided wherever the alignment of the range allows.
int plan_z_segments(const Run& r, Plan& plan, int& ns, unsigned long long& cur, unsigned long long& units,
                    unsigned long long to, bool taper)
{
    const int zu = ZB + 7;                                              // unit bits at Lw = 0
    int Lw = floor_log2(to - cur) - zu - 11;                            // about 2^11 units: several waves of CTAs
    const int lw_floor = r.lw_max < 5 ? r.lw_max : 5;
    Lw = Lw < lw_floor ? lw_floor : (Lw > r.lw_max ? r.lw_max : Lw);
    while (cur < to) {
        const unsigned long long left = to - cur;
        while (Lw > 0 && ((cur & ((1ull << (zu + Lw)) - 1ull)) || (left >> (zu + Lw)) == 0)) --Lw;
        unsigned long long sz = left >> (zu + Lw) << (zu + Lw);
        if (Lw > lw_floor && taper) sz = (left - (left >> 3)) >> (zu + Lw) << (zu + Lw);
        const unsigned long long nu = sz >> (zu + Lw);
        if (nu) {
            if (ns >= MAX_SEGMENTS) { t_last_error = "internal: bad work plan"; return ISING_ERR_INTERNAL; }
            plan.seg[ns] = Segment{cur, units, nu, 0ull, zu + Lw, 0};
            units += nu;
            cur += nu << (zu + Lw);
            ++ns;
        } else if (Lw == 0) {
            t_last_error = "internal: range not aligned for the tensor-core screen";
            return ISING_ERR_INTERNAL;
        }
        if (cur < to) {
            const int next = Lw > lw_floor + 3 ? Lw - 3 : lw_floor;
            Lw = next < Lw ? next : (Lw > 0 ? Lw - 1 : 0);                 // below the floor only to finish a ragged end
        }
    }
    return ISING_OK;
}

// ---- single-pass path: the whole range in one to three launches without host decisions in between (except the
// one described below), threshold refreshed on the device, then compaction and the one-block final selection.
// Ranges of 2^z_min_log2 states and more: the bulk goes through the tensor-core screen (zscreen.cu) -- the packed
// kernel ramps the threshold up over the first 2^34 states (or an eighth of the range), the next stretch of the same
// size is a PROBE of the screen, and only if fewer than 1 in 48 of its blocks were flagged (an instance whose table
// range forces a blunt lambda, or a spectrum dense at the bottom, fails this) does the rest follow the same way;
// otherwise the packed kernel finishes. Returns ISING_OK with *redo = true if the candidate pool overflowed. ----
int run_single_pass(Run& r, unsigned long long* states_out, double* energies_out, bool* redo)
{
    Workspace& ws = *r.ws;
    *redo = false;
    Plan plan;
    plan_header(r, plan, 1, INT32_MIN);
    const unsigned long long range = r.q_end - r.q_begin;
    const bool direct = r.N <= N_DIRECT_MAX;
    // The screen's units are 2^21 states, aligned; range bounds are multiples of 2^20 only (include/ising.h). A ragged
    // head (q_begin an odd multiple of 2^20) is absorbed by the packed ramp-up, which then ends at the next multiple
    // of 2^21; a ragged tail [z_end, q_end) of 2^20 states follows the bulk launch through the packed kernel.
    const unsigned long long zmask = (1ull << (ZB + 7)) - 1ull;
    const bool use_z = !direct && (r.variant == 0 || r.variant == 128) && range >= (1ull << r.z_min_log2) &&
                       range >= (1ull << (ZB + 7 + 3));
    const unsigned long long z_end = r.q_end & ~zmask;                    // end of the screen's stretch
    int rc = ISING_OK;
    auto timed_launch = [&](auto&& launch) -> int {
        CUDA_TRY(cudaEventRecord(ws.ev[2], r.st));
        const int lrc = launch();
        if (lrc != ISING_OK) return lrc;
        CUDA_TRY(cudaEventRecord(ws.ev[3], r.st));
        return ISING_OK;
    };
    bool last_was_z = false;
    unsigned long long last_z_configs = 0;
    auto add_elapsed = [&]() -> int {
        float ms = 0.f;
        CUDA_TRY(cudaEventElapsedTime(&ms, ws.ev[2], ws.ev[3]));
        r.enum_ms += ms;
        if (last_was_z) { r.z_ms += ms; r.z_configs += last_z_configs; }
        last_was_z = false;
        return ISING_OK;
    };
    if (direct) {
        rc = timed_launch([&]() -> int {
            launch_direct(ws.tab, ws.ctrl, ws.pool, ws.hist, r.N, r.S, (unsigned)range, 1, r.st);
            LAUNCH_CHECK("direct_kernel");
            r.stats->kernel_launches += 1;
            r.stats->enum_launches += 1;
            return ISING_OK;
        });
        if (rc != ISING_OK) return rc;
    } else {
        // a2': the first X states are formed exactly, one 1024-configuration block per warp -- 2^15 of them without any
        // threshold, the rest under the threshold those give (which most blocks would pass anyway; X shrinks with S so
        // that the candidates of this phase, about X S / 2^15, stay far below the pool size). Then walked segments.
        const unsigned long long prime = 1ull << MIN_CHUNK_BITS;
        unsigned long long X = 1ull << 21;
        while (X > prime && X * (unsigned long long)r.S > (1ull << 35)) X >>= 1;
        if (X > range) X = range;
        unsigned long long p0 = range;                                   // end of the packed kernel's stretch
        if (use_z) { p0 = 1ull << r.z_ramp_log2; while (p0 > range / 8) p0 >>= 1; }       // 2^21 <= p0 <= range / 8
        // states [q_begin, ramp_end) go through the packed kernel, [ramp_end, probe_end) are the probe of the screen
        const unsigned long long ramp_end = use_z ? (r.q_begin + p0 + zmask) & ~zmask : r.q_end;
        const unsigned long long probe_end = ramp_end + p0;               // <= z_end because range >= 8 p0 >= 2^24
        int ns = 0;
        unsigned long long cur = r.q_begin, units = 0;
        plan.seg[ns++] = Segment{cur, units, prime >> LOWBITS, 0ull, LOWBITS, 0};
        units += prime >> LOWBITS; cur += prime;
        if (X > prime) {
            plan.seg[ns++] = Segment{cur, units, (X - prime) >> LOWBITS, prime, LOWBITS, 0};
            units += (X - prime) >> LOWBITS; cur += X - prime;
        }
        rc = plan_walk_segments(r, plan, ns, cur, units, ramp_end, prime);
        if (rc != ISING_OK) return rc;
        plan.nseg = ns;
        plan.total_units = units;
        rc = timed_launch([&]() -> int { return launch_walk(r, plan); });
        if (rc != ISING_OK) return rc;
        if (use_z) {
            launch_ztables(ws.tab, ws.ctrl, ws.zt, r.N, r.st);
            LAUNCH_CHECK("ztables_kernel");
            // ---- probe: the next p0 states through the tensor-core screen ----
            reset_queue_kernel<<<1, 1, 0, r.st>>>(ws.ctrl, 0);
            Plan zp;
            plan_header(r, zp, 1, INT32_MIN);
            ns = 0; units = 0;
            rc = plan_z_segments(r, zp, ns, cur, units, probe_end, false);
            if (rc != ISING_OK) return rc;
            zp.nseg = ns; zp.total_units = units;
            CUDA_TRY(cudaEventRecord(ws.ev[3], r.st));                   // (the ramp-up launch ends here)
            rc = read_ctrl(r);                                           // ... and is timed while the probe is enqueued
            if (rc != ISING_OK) return rc;
            if ((rc = add_elapsed()) != ISING_OK) return rc;
            if (ws.h_ctrl->status != ISING_OK) return ISING_OK;
            rc = timed_launch([&]() -> int { return launch_z(r, zp); });
            if (rc != ISING_OK) return rc;
            r.stats->kernel_launches += 3;
            r.stats->enum_launches += 1;
            r.stats->z_launches += 1;
            last_was_z = true;
            last_z_configs = probe_end - ramp_end;
            rc = read_ctrl(r);
            if (rc != ISING_OK) return rc;
            if ((rc = add_elapsed()) != ISING_OK) return rc;
            const double zs = (double)ws.h_ctrl->z_steps, zf = (double)ws.h_ctrl->z_flagged;
            // Cost model behind the constant 48: a clean step (128 blocks, one per thread) takes 1.8 us and the packed
            // kernel is 14 times slower, i.e. 25 us for the same 2^21 states; a flagged block takes its WARP about 20 us.
            // If the flagged blocks of a step spread evenly over the CTA's four warps the screen breaks even at about
            // 1 flagged block in 27, if they all fall to one warp at 1 in 109. 1 in 48 sits between the two and is
            // the rate up to which the screen was measured to win (N = 42, S = 65536: 22 ms against 135 ms). The probe
            // runs under the loosest threshold of the bulk, but it is only a sample: an instance whose low states cluster
            // late in q order can flag more often later on. That costs time, never a state.
            // ISING_Z_FORCE = 1 (tests): the bulk takes the screen whatever the probe flagged, so that the flagged-block
            // path is compared with the oracle under load.
            const bool z_ok = !ws.h_ctrl->pool_overflow && zs > 0.0 && (r.z_force || zf * 48.0 <= zs);
            reset_queue_kernel<<<1, 1, 0, r.st>>>(ws.ctrl, 0);
            r.stats->kernel_launches += 1;
            Plan rest;
            plan_header(r, rest, 1, INT32_MIN);
            ns = 0; units = 0;
            Plan tail;                                                   // z_ok and a ragged end: [z_end, q_end), packed kernel
            plan_header(r, tail, 1, INT32_MIN);
            if (z_ok) {
                rc = plan_z_segments(r, rest, ns, cur, units, z_end, true);
                r.stats->kernel_variant = 128;
                if (rc == ISING_OK && z_end < r.q_end) {
                    tail.seg[0] = Segment{z_end, 0ull, (r.q_end - z_end) >> MIN_CHUNK_BITS, 0ull, MIN_CHUNK_BITS, 0};
                    tail.nseg = 1;
                    tail.total_units = tail.seg[0].n_units;
                    cur = r.q_end;
                }
            } else {
                rc = plan_walk_segments(r, rest, ns, cur, units, r.q_end, 0ull);
            }
            if (rc != ISING_OK) return rc;
            rest.nseg = ns; rest.total_units = units;
            if (cur != r.q_end) { t_last_error = "internal: work plan does not cover the range"; return ISING_ERR_INTERNAL; }
            rc = timed_launch([&]() -> int {
                if (!z_ok) return launch_walk(r, rest);
                const int zrc = launch_z(r, rest);
                if (zrc != ISING_OK) return zrc;
                r.stats->kernel_launches += 1;
                r.stats->enum_launches += 1;
                r.stats->z_launches += 1;
                if (tail.nseg) {
                    reset_queue_kernel<<<1, 1, 0, r.st>>>(ws.ctrl, 0);
                    r.stats->kernel_launches += 1;
                    return launch_walk(r, tail);
                }
                return ISING_OK;
            });
            if (rc != ISING_OK) return rc;
            if (z_ok) { last_was_z = true; last_z_configs = z_end - probe_end; }
        } else if (cur != r.q_end) {
            t_last_error = "internal: work plan does not cover the range";
            return ISING_ERR_INTERNAL;
        }
    }
    r.stats->kernel_launches += launch_compact(ws.pool, ws.pool2, ws.ctrl, plan, r.st);
    LAUNCH_CHECK("compact_kernel");
    r.stats->kernel_launches += launch_final_small(r.mode ? r.Jorig : r.J, r.mode ? r.horig : r.h, r.N, r.mode, ws.pool2,
                                                   ws.ctrl, r.S, r.keep_cap, states_out, energies_out, r.st);
    LAUNCH_CHECK("final_small_kernel");
    CUDA_TRY(cudaEventRecord(ws.ev[1], r.st));          // end of the call if the one-block selection sufficed
    rc = read_ctrl(r);
    if (rc != ISING_OK) return rc;
    if ((rc = add_elapsed()) != ISING_OK) return rc;
    const Ctrl& c = *ws.h_ctrl;
    if (c.status != ISING_OK) return ISING_OK;          // rejected by the staging kernel: the caller reports it
    r.stats->configs += range;
    if (c.pool_overflow) { *redo = true; return ISING_OK; }
    r.stats->candidates += c.count;
    r.stats->z_blocks = c.z_steps;
    r.stats->z_flagged_blocks = c.z_flagged;
    if (c.final_state == 1) { r.stats->keep = (int)c.kept; r.done = true; return ISING_OK; }
    if (c.final_state != 2 || c.count2 < (unsigned)r.S) {
        t_last_error = "internal: fewer candidates than requested states";
        return ISING_ERR_INTERNAL;
    }
    // many candidates (large S): the general multi-block selection on the compacted pool
    r.stats->kernel_launches += launch_select(ws.pool2, ws.ctrl, c.count2, r.S, plan, r.st);
    LAUNCH_CHECK("select kernels");
    rc = read_ctrl(r);
    if (rc != ISING_OK) return rc;
    if (ws.h_ctrl->band_overflow) {
        // the kept list was cut: bring the cut list to `pool`, where the band pass expects it
        copy_entries_kernel<<<(ws.h_ctrl->kept + 255) / 256, 256, 0, r.st>>>(ws.pool2, ws.pool, ws.h_ctrl->kept);
        LAUNCH_CHECK("copy_entries_kernel");
        r.stats->kernel_launches += 1;
        return ISING_OK;
    }
    r.stats->keep = (int)ws.h_ctrl->kept;
    r.stats->kernel_launches += launch_final(r.mode ? r.Jorig : r.J, r.mode ? r.horig : r.h, r.N, r.mode, ws.pool2,
                                             ws.h_ctrl->kept, r.S, states_out, energies_out, r.st);
    LAUNCH_CHECK("final kernels");
    return ISING_OK;
}

struct Piece {
    unsigned long long base;
    unsigned long long n_units;
    int unit_bits;
};

// ---- host-sequenced path: the range in pieces, a selection (normal mode) or an fp64 drain (band mode) after every
// piece, a piece whose candidates overflow the pool re-run in halves. Used when the single pass was void (adversarial
// orderings, very large S late in the spectrum) and for the band pass. Leaves the kept list in pool[0..kept). ----
int run_pieces(Run& r, bool band_mode, int loE, unsigned want)
{
    Workspace& ws = *r.ws;
    Plan plan;
    plan_header(r, plan, 0, band_mode ? loE : INT32_MIN);
    plan.nseg = 1;
    unsigned long long cur = r.q_begin, processed = 0;
    std::vector<Piece> stack;
    bool tau_finite = band_mode;
    while (cur < r.q_end || !stack.empty()) {
        Piece pc;
        if (!stack.empty()) {
            pc = stack.back();
            stack.pop_back();
        } else if (r.N <= N_DIRECT_MAX) {
            pc = Piece{cur, (r.q_end - cur) >> (r.N < LOWBITS ? r.N : LOWBITS), r.N < LOWBITS ? r.N : LOWBITS};
            cur = r.q_end;
        } else if (processed == 0 && !band_mode) {
            pc = Piece{cur, 1ull << (MIN_CHUNK_BITS - LOWBITS), LOWBITS};      // a2': formed exactly
            cur += 1ull << MIN_CHUNK_BITS;
        } else {
            const unsigned long long remaining = r.q_end - cur;
            unsigned long long target = band_mode ? (1ull << r.chunk_log2) : (unsigned long long)r.growth * processed;
            if (target > (1ull << r.chunk_log2)) target = 1ull << r.chunk_log2;
            if (!tau_finite && target > (1ull << 16)) target = 1ull << 16;     // everything passes: keep it small
            if (target < (1ull << MIN_CHUNK_BITS)) target = 1ull << MIN_CHUNK_BITS;
            const unsigned long long sz = target < remaining ? target : remaining;
            const int Lw = choose_lw(cur, sz, r.lw_max);
            pc = Piece{cur, sz >> (MIN_CHUNK_BITS + Lw), MIN_CHUNK_BITS + Lw};
            if (pc.n_units == 0) { t_last_error = "internal: bad launch plan"; return ISING_ERR_INTERNAL; }
            cur += pc.n_units << pc.unit_bits;
        }
        const unsigned long long pc_size = pc.n_units << pc.unit_bits;
        if (r.N <= N_DIRECT_MAX) {
            // tiny instance: everything at once through the direct kernel (its 2^N states always fit)
            launch_direct(ws.tab, ws.ctrl, ws.pool, ws.hist, r.N, r.S, (unsigned)(r.q_end - r.q_begin), 0, r.st);
            LAUNCH_CHECK("direct_kernel");
            r.stats->kernel_launches += 1;
            r.stats->enum_launches += 1;
        } else {
            plan.seg[0] = Segment{pc.base, 0ull, pc.n_units, 0ull, pc.unit_bits, 0};
            plan.total_units = pc.n_units;
            plan.q_end = r.q_end;
            reset_queue_kernel<<<1, 1, 0, r.st>>>(ws.ctrl, 0);
            CUDA_TRY(cudaEventRecord(ws.ev[2], r.st));
            int rc = launch_walk(r, plan);
            if (rc != ISING_OK) return rc;
            CUDA_TRY(cudaEventRecord(ws.ev[3], r.st));
            r.stats->kernel_launches += 1;
        }
        int rc = read_ctrl(r);
        if (rc != ISING_OK) return rc;
        if (r.N > N_DIRECT_MAX) {
            float ms = 0.f;
            CUDA_TRY(cudaEventElapsedTime(&ms, ws.ev[2], ws.ev[3]));
            r.enum_ms += ms;
        }
        const unsigned count = ws.h_ctrl->count, kept = ws.h_ctrl->kept;
        if (ws.h_ctrl->pool_overflow) {
            // pool overflow: drop this piece's candidates and run it again in two halves
            reset_queue_kernel<<<1, 1, 0, r.st>>>(ws.ctrl, 1);
            r.stats->kernel_launches += 1;
            r.stats->split_retries += 1;
            Piece a = pc, b = pc;
            if (pc.n_units >= 2) {
                a.n_units = pc.n_units / 2;
                b.n_units = pc.n_units - a.n_units;
                b.base = pc.base + (a.n_units << pc.unit_bits);
            } else if (pc.unit_bits > MIN_CHUNK_BITS) {
                a.unit_bits = b.unit_bits = pc.unit_bits - 1;
                a.n_units = b.n_units = 1;
                b.base = pc.base + (1ull << a.unit_bits);
            } else {
                t_last_error = "internal: candidate pool overflow on a minimal launch";
                return ISING_ERR_INTERNAL;
            }
            stack.push_back(b);
            stack.push_back(a);
            continue;
        }
        processed += pc_size;
        r.stats->configs += pc_size;
        r.stats->candidates += count - kept;
        if (band_mode) {
            if (count > kept)
                r.stats->kernel_launches += launch_band_drain(r.mode ? r.Jorig : r.J, r.mode ? r.horig : r.h, r.N, r.mode,
                                                              ws.pool, ws.ctrl, kept, count, want, r.st);
        } else if (count > kept) {
            r.stats->kernel_launches += launch_select(ws.pool, ws.ctrl, count, r.S, plan, r.st);
            if (count >= (unsigned)r.S) tau_finite = true;
        }
        LAUNCH_CHECK("selection kernels");
    }
    return read_ctrl(r);
}

// mode 0: (J, h) is an Ising instance, energies by eq. (1). mode 1: (Jorig, horig) = QUBO (a, b); (J, h) its Ising image.
int run_lowest(const double* J, const double* h, const double* Jorig, const double* horig, int mode, double extra_eps_rel,
               int N, int S, unsigned long long q_begin, unsigned long long q_end,
               unsigned long long* states_out, double* energies_out, cudaStream_t st)
{
    Workspace& ws = t_ws;
    ising_stats stats;
    memset(&stats, 0, sizeof(stats));
    Run r;
    r.ws = &ws; r.stats = &stats;
    r.J = J; r.h = h; r.Jorig = Jorig; r.horig = horig;
    r.mode = mode; r.N = N; r.S = S;
    r.lw_max = env_int("ISING_LW", LW_MAX, 0, LW_MAX);
    r.chunk_log2 = env_int("ISING_CHUNK_LOG2", 42, MIN_CHUNK_BITS, 44);
    r.growth = env_int("ISING_GROWTH", 3, 1, 1 << 20);      // a segment is at most growth x what lies before it
    // 0 (default): packed 16-bit screen, plus the tensor-core screen for the bulk of large ranges; 16: packed screen only;
    // 32: int32 kernel only; 128: as 0
    const int kv = env_int("ISING_KERNEL", 0, 0, 128);
    r.variant = kv == 32 ? 32 : (kv == 16 ? 16 : 0);
    r.z_min_log2 = env_int("ISING_Z_MIN_LOG2", 36, ZB + 10, 63);
    r.z_ramp_log2 = env_int("ISING_Z_RAMP_LOG2", 34, ZB + 7, 44);
    r.z_force = env_int("ISING_Z_FORCE", 0, 0, 1);
    // test knob for the band pass: a selection keeps at most 2^k entries (never fewer than S)
    r.keep_cap = 1u << env_int("ISING_KEEP_CAP_LOG2", 20, 5, 20);
    while (r.keep_cap < (unsigned)S) r.keep_cap <<= 1;
    const int path = env_int("ISING_PATH", 0, 0, 1);        // 1: skip the single pass (tests of the host-sequenced path)
    r.q_begin = q_begin; r.q_end = q_end; r.st = st; r.enum_ms = 0.0; r.z_ms = 0.0; r.z_configs = 0; r.done = false;
    const int rb = floor_log2(q_end - q_begin - 1) + 1;     // bits of the range
    r.qshift = rb > 31 ? rb - 31 : 0;                       // (range >> qshift) < 2^32 - 1

    CUDA_TRY(cudaEventRecord(ws.ev[0], st));
    launch_stage(J, h, N, ws.tab, ws.ctrl, ws.hist, st, extra_eps_rel);
    LAUNCH_CHECK("stage_kernel");
    stats.kernel_launches += 1;
    stats.inner_bits = LOWBITS;
    stats.kernel_variant = r.variant == 32 ? 32 : 16;      // 128 once the tensor-core screen took the bulk
    stats.passes = 1;

    bool redo = (path == 1);
    int rc = ISING_OK;
    if (!redo) {
        rc = run_single_pass(r, states_out, energies_out, &redo);
        if (rc != ISING_OK) return rc;
    } else {
        rc = read_ctrl(r);
        if (rc != ISING_OK) return rc;
    }
    if (ws.h_ctrl->status != ISING_OK) {
        t_last_error = std::string("instance rejected: ") + ising_strerror(ws.h_ctrl->status);
        return ws.h_ctrl->status;
    }
    stats.grid_exponent = ws.h_ctrl->p;
    stats.exact = ws.h_ctrl->exact;
    stats.epsilon = ws.h_ctrl->epsilon;
    stats.screen_shift = r.variant != 32 ? ws.h_ctrl->shift16 : -1;
    const int band = ws.h_ctrl->band;

    if (redo) {
        // the single pass was void (or skipped): the same range again, host-sequenced
        if (path == 0) {
            stats.passes += 1; stats.configs = 0; stats.candidates = 0;
            stats.z_blocks = stats.z_flagged_blocks = 0; stats.z_launches = 0; r.z_ms = 0.0; r.z_configs = 0;
        }
        restart_kernel<<<1, 1, 0, st>>>(ws.ctrl, tau_pack(TAU_INF, QC_NONE));
        LAUNCH_CHECK("restart_kernel");
        stats.kernel_launches += 1;
        rc = run_pieces(r, false, 0, 0);
        if (rc != ISING_OK) return rc;
        if (!ws.h_ctrl->band_overflow) {
            const unsigned kept = ws.h_ctrl->kept;
            if (kept < (unsigned)S) { t_last_error = "internal: fewer states kept than requested"; return ISING_ERR_INTERNAL; }
            stats.keep = (int)kept;
            stats.kernel_launches += launch_final(mode ? Jorig : J, mode ? horig : h, N, mode, ws.pool, kept, S,
                                                  states_out, energies_out, st);
            LAUNCH_CHECK("final kernels");
        }
    }
    if (ws.h_ctrl->band_overflow) {
        // ---- G3 fallback: more than KEEP_CAP states lie within the guard band of the S-th
        // lowest grid energy eS, so the band cannot be kept resident. Every state with grid energy < eS - band is
        // certainly among the S lowest (they are a sorted prefix of the kept list); the others come from the states
        // with grid energy in [eS - band, eS + band], which a second enumeration streams through the pool: each
        // piece's band states are re-evaluated in fp64 and merged into the running best S - n_sure under (E64, q).
        const unsigned kept = ws.h_ctrl->kept;
        const int eS = ws.h_ctrl->eS;
        count_sure_kernel<<<1, 32, 0, st>>>(ws.pool, ws.ctrl, kept, band);
        LAUNCH_CHECK("count_sure_kernel");
        rc = read_ctrl(r);
        if (rc != ISING_OK) return rc;
        const unsigned n_sure = ws.h_ctrl->n_sure;
        if (n_sure >= (unsigned)S) { t_last_error = "internal: band pass bookkeeping"; return ISING_ERR_INTERNAL; }
        if (n_sure) {
            copy_entries_kernel<<<(n_sure + 255) / 256, 256, 0, st>>>(ws.pool, ws.pool2, n_sure);
            LAUNCH_CHECK("copy_entries_kernel");
        }
        const long long hi = (long long)eS + band;
        restart_kernel<<<1, 1, 0, st>>>(ws.ctrl, tau_pack(hi < (long long)TAU_INF ? (int)hi : TAU_INF, QC_NONE));
        LAUNCH_CHECK("restart_kernel");
        stats.kernel_launches += 3;
        stats.passes += 1;
        const unsigned want = (unsigned)S - n_sure;
        rc = run_pieces(r, true, eS - band, want);
        if (rc != ISING_OK) return rc;
        if (ws.h_ctrl->kept < want) { t_last_error = "internal: band pass found too few states"; return ISING_ERR_INTERNAL; }
        // final list = sure states + best band states: pool2[0..n_sure) + pool[0..want), all re-evaluated in fp64
        copy_entries_kernel<<<(want + 255) / 256, 256, 0, st>>>(ws.pool, ws.pool2 + n_sure, want);
        LAUNCH_CHECK("copy_entries_kernel");
        stats.keep = S;
        stats.kernel_launches += 1 + launch_final(mode ? Jorig : J, mode ? horig : h, N, mode, ws.pool2, (unsigned)S, S,
                                                  states_out, energies_out, st);
        LAUNCH_CHECK("final kernels");
    }
    if (!r.done) {
        CUDA_TRY(cudaEventRecord(ws.ev[1], st));
        CUDA_TRY(cudaStreamSynchronize(st));
    }
    CUDA_TRY(cudaGetLastError());
    float total_ms = 0.f;
    CUDA_TRY(cudaEventElapsedTime(&total_ms, ws.ev[0], ws.ev[1]));
    stats.enum_ms = r.enum_ms;
    stats.total_ms = total_ms;
    stats.z_ms = r.z_ms;
    stats.z_configs = r.z_configs;
    stats.hit_blocks = ws.h_ctrl->hits;
    stats.false_hit_blocks = ws.h_ctrl->false_hits;
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

void set_last_error(const char* what) { t_last_error = what ? what : ""; }

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
    launch_stage(J_dev, h_dev, N, ws.tab, ws.ctrl, nullptr, st, 0.0);
    stats.kernel_launches += 1;
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
    launch_stage(J_dev, h_dev, N, ws.tab, ws.ctrl, nullptr, st, 0.0);          // validation only (same error codes)
    stats.kernel_launches += 1;
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

int ising_addmin_mix_peak(double ms_target, double* addmin_per_s_out_host, void* stream)
{
    if (!addmin_per_s_out_host) return ISING_ERR_NULL;
    double r = run_fma_peak(ms_target, (cudaStream_t)stream, 3);
    if (r < 0.0) { t_last_error = "add-min mix microbenchmark failed"; return ISING_ERR_CUDA; }
    *addmin_per_s_out_host = r;
    return ISING_OK;
}

int ising_zscreen_selftest(uint32_t seed, double* rel_under_out_host, double* rel_over_out_host, void* stream)
{
    t_last_error.clear();
    if (!rel_under_out_host || !rel_over_out_host) { t_last_error = "null pointer argument"; return ISING_ERR_NULL; }
    int rc = ensure_workspace();
    if (rc != ISING_OK) return rc;
    cudaStream_t st = (cudaStream_t)stream;
    double* d = t_ws.out_e;                                  // two doubles of the output staging buffer
    launch_zselftest(seed, d, st);
    LAUNCH_CHECK("zselftest_kernel");
    double h[2] = {0.0, 0.0};
    CUDA_TRY(cudaMemcpyAsync(h, d, sizeof(h), cudaMemcpyDeviceToHost, st));
    CUDA_TRY(cudaStreamSynchronize(st));
    *rel_under_out_host = h[0];
    *rel_over_out_host = h[1];
    return ISING_OK;
}

void ising_release_workspace(void) { if (t_ws.device >= 0) t_ws.release(); }

}  // extern "C"
