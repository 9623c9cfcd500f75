// walk.cuh -- the persistent enumeration kernel (SURVEY.md section 8 rows a2, a2', a3, a4 and the publishing half of
// a5), shared by the packed 16-bit screen (enumerate16.cu) and the int32 variant (enumerate.cu).
//
// One launch enumerates a whole state range. Every WARP is a worker: it takes ONE unit from the queue in Ctrl
// (ascending q), builds the base state of the unit (a2), walks it (a3), screens every 1024-configuration block
// against the threshold tau (a4) and forms the blocks that pass exactly (int32) to push the survivors to the pool;
// the grid has one warp per unit. (A persistent loop over units inside the kernel was measured and dropped: with the
// back edge around the Gray loop ptxas no longer finds a register allocation in which the three sources of every
// add-min sit in different banks -- 63 of 440 conflict, 6 % in throughput -- whereas this form has none.)
//
// tau is refreshed ON THE DEVICE (north_star (b): "running S-th-best energy broadcast from global memory"): every
// pushed candidate is also counted in a two-level histogram of grid energies in global memory, and the warp whose
// push makes the pool count cross a multiple of Plan::refresh scans the histogram for the lowest bin edge b with at
// least S candidates at or below it. Counts only grow and every counted candidate is a distinct configuration, so
// "S configurations have grid energy <= b" holds from then on and  tauE = b + band  can never cut a state of the
// final list; it is published with one atomicMin on the 64-bit threshold word and re-read by
// every warp at the start of a unit and every 16 Gray steps. For exact instances the word also carries a limit on q
// for ties on tauE: the next state the queue had not handed out when the histogram was scanned -- every counted
// candidate lies below it, so a later configuration that merely ties on tauE cannot enter the list.
//
// Ramp-up (a2'): the first segments are formed exactly, one 1024-configuration block per warp (no threshold exists
// yet, then a poor one under which most blocks would pass the screen anyway), the following segments double in
// size, and a unit of a segment starts only when Segment::need_done configurations are complete, so that the
// threshold it starts with is never older than about half of the states before it. The wait cannot deadlock: a
// warp only ever waits for units that were handed out before its own, i.e. to warps that are already running.
#pragma once
#include "common.cuh"

namespace ising {

__device__ __forceinline__ unsigned long long ld_relaxed_u64(const unsigned long long* p)
{
    unsigned long long v;
    asm volatile("ld.relaxed.gpu.global.u64 %0, [%1];" : "=l"(v) : "l"(p) : "memory");
    return v;
}
__device__ __forceinline__ unsigned ld_relaxed_u32(const unsigned* p)
{
    unsigned v;
    asm volatile("ld.relaxed.gpu.global.u32 %0, [%1];" : "=r"(v) : "l"(p) : "memory");
    return v;
}

// First state of queue unit u (plan.q_end if the queue is exhausted).
__device__ inline unsigned long long unit_to_q(const Plan& plan, unsigned long long u)
{
    if (u >= plan.total_units) return plan.q_end;
    int s = 0;
    while (s + 1 < plan.nseg && u >= plan.seg[s].first_unit + plan.seg[s].n_units) ++s;
    return plan.seg[s].q0 + ((u - plan.seg[s].first_unit) << plan.seg[s].unit_bits);
}

// Warp-collective: first index i in [0, 256) with  sum_{j <= i} h[j] >= target, and the sum before it; -1 if the
// 256 counters hold fewer than target. Lane l reads h[8 l .. 8 l + 7].
__device__ inline int scan256(const unsigned* h, unsigned target, unsigned& before, int lane)
{
    unsigned c[8], sum = 0;
#pragma unroll
    for (int k = 0; k < 8; ++k) { c[k] = ld_relaxed_u32(h + lane * 8 + k); sum += c[k]; }
    unsigned incl = sum;
#pragma unroll
    for (int d = 1; d < 32; d <<= 1) {
        const unsigned n = __shfl_up_sync(0xffffffffu, incl, d);
        if (lane >= d) incl += n;
    }
    const unsigned ball = __ballot_sync(0xffffffffu, incl >= target);
    if (!ball) return -1;
    const int src = __ffs(ball) - 1;
    unsigned cum = incl - sum;
    int kk = 0;
    if (lane == src)
        while (kk < 7 && cum + c[kk] < target) { cum += c[kk]; ++kk; }
    before = __shfl_sync(0xffffffffu, cum, src);
    return __shfl_sync(0xffffffffu, lane * 8 + kk, src);
}

// Warp-collective: the lowest threshold the candidate histogram certifies -- the upper edge of the first bin with at
// least S candidates at or below it, plus the guard band. false: fewer than S candidates so far.
__device__ inline bool hist_threshold(const Ctrl* __restrict__ ctrl, const unsigned* __restrict__ hist, unsigned S,
                                      int lane, int& tauE)
{
    unsigned before = 0, before2 = 0;
    const int coarse = scan256(hist, S, before, lane);
    if (coarse < 0) return false;
    int fine = scan256(hist + HIST_COARSE + coarse * 256, S - before, before2, lane);
    if (fine < 0) fine = 255;                                  // coarse and fine counters are updated separately
    const long long bin = (long long)coarse * 256 + fine;
    const long long edge = -ctrl->Wq + ((bin + 1) << ctrl->hist_shift) - 1 + ctrl->band;
    tauE = edge < (long long)TAU_INF ? (int)edge : TAU_INF;
    return true;
}

// Warp-collective: derive a threshold from the candidate histogram and publish it (see the file header).
static __device__ __noinline__ void refresh_tau(Ctrl* __restrict__ ctrl, const unsigned* __restrict__ hist, const Plan& plan,
                                         int lane)
{
    int tauE;
    if (!hist_threshold(ctrl, hist, (unsigned)plan.S, lane, tauE)) return;
    unsigned qc = QC_NONE;
    if (ctrl->exact) {
        __threadfence();                                       // every candidate counted above came from a unit < nu
        const unsigned long long nu = ld_relaxed_u64(&ctrl->next_unit);
        const unsigned long long d = unit_to_q(plan, nu) - plan.q_begin;
        const unsigned long long v = (d + ((1ull << plan.qshift) - 1ull)) >> plan.qshift;     // rounded up: looser
        qc = v < (unsigned long long)QC_NONE ? (unsigned)v : QC_NONE;
    }
    if (lane == 0) atomicMin(&ctrl->tau, tau_pack(tauE, qc));
}

// Histogram bin of a grid energy (fine bin; coarse bin = fine >> 8).
__device__ __forceinline__ int hist_bin(int e, long long Wq, int hist_shift)
{
    long long b = ((long long)e + Wq) >> hist_shift;
    return b < 0 ? 0 : (b >= HIST_FINE ? HIST_FINE - 1 : (int)b);
}

// Warp-collective local fields of the spins i = lane and i = lane + 32 at state q, and the grid energy of q:
//   Phi_i(q) = hq_i + sum_j Jq_ij s_j(q) ,   E(q) = -1/2 sum_i s_i (Phi_i + hq_i)      (eq. (1))
__device__ __forceinline__ int warp_fields(const Tables* __restrict__ tab, int N, unsigned long long q, int lane,
                                           int& phi_lo, int& phi_hi)
{
    const int* __restrict__ Jq = tab->Jq;
    int a0 = 0, a1 = 0;
    for (int j = 0; j < N; ++j) {
        const bool up = (q >> j) & 1ull;
        const int v0 = Jq[j * 64 + lane], v1 = Jq[j * 64 + lane + 32];        // row j = column j (symmetric): coalesced
        a0 += up ? v0 : -v0;
        a1 += up ? v1 : -v1;
    }
    const int h0 = tab->hq[lane], h1 = tab->hq[lane + 32];                   // entries >= N are zero
    phi_lo = a0 + h0;
    phi_hi = a1 + h1;
    int part = ((q >> lane) & 1ull) ? (phi_lo + h0) : -(phi_lo + h0);
    part += ((q >> (lane + 32)) & 1ull) ? (phi_hi + h1) : -(phi_hi + h1);
    return -(__reduce_add_sync(0xffffffffu, part) / 2);                      // the sum is even
}

// a4, second half: the whole warp forms the 1024 energies of one block exactly (int32 grid units) and pushes the
// survivors. qh = the block's state with lo and mid bits zero, eh = its grid energy (FROM_SCRATCH: computed here).
// Kept out of line so that its registers do not weigh on the enumeration loop.
template <bool FROM_SCRATCH>
__device__ __noinline__ void form_block(const Tables* __restrict__ tab, Ctrl* __restrict__ ctrl,
                                        Entry* __restrict__ pool, unsigned* __restrict__ hist, const Plan& plan,
                                        const int* sC, unsigned long long qh, int eh, unsigned long long tau, int lane)
{
    const int N = plan.N;
    int vx = tab->QL[lane], ux = tab->QM[lane];
    if (FROM_SCRATCH) {
        int plo, phi_unused;
        eh = warp_fields(tab, N, qh, lane, plo, phi_unused);
#pragma unroll
        for (int i = 0; i < LOWBITS; ++i) {
            const int f = __shfl_sync(0xffffffffu, plo, i);
            if (i < LL) { if (lane >> i & 1) vx -= 2 * f; }
            else        { if (lane >> (i - LL) & 1) ux -= 2 * f; }
        }
    } else {
        const int* __restrict__ Jq = tab->Jq;
        for (int i = 0; i < LOWBITS; ++i) {
            // local field of spin i at the block's state, summed by the warp
            int part = 0;
            for (int j = lane; j < N; j += 32) {
                const int w = Jq[i * 64 + j];
                part += ((qh >> j) & 1ull) ? w : -w;
            }
            const int f = tab->hq[i] + __reduce_add_sync(0xffffffffu, part);
            if (i < LL) { if (lane >> i & 1) vx -= 2 * f; }
            else        { if (lane >> (i - LL) & 1) ux -= 2 * f; }
        }
    }
    const int tauE = tau_energy(tau);
    const unsigned qc = tau_qc(tau);
    const unsigned long long tauQ = qc == QC_NONE ? Q_MAX : plan.q_begin + ((unsigned long long)qc << plan.qshift);
    const int loE = plan.loE;
    const unsigned long long qs = qh + (unsigned)lane;
    const int v = vx + eh;
    // two passes: mark the survivors, reserve their pool slots with ONE atomic per block, then write
    unsigned mask = 0;
    for (int mid = 0; mid < NMID; ++mid) {
        const int e = v + sC[mid * NLO + lane] + __shfl_sync(0xffffffffu, ux, mid);
        const unsigned long long q = qs + ((unsigned)mid << LL);
        const bool pass = (e < tauE || (e == tauE && q < tauQ)) && e >= loE && q < plan.q_end;
        mask |= pass ? (1u << mid) : 0u;
    }
    const int cnt = __popc(mask);
    int incl = cnt;
#pragma unroll
    for (int d = 1; d < 32; d <<= 1) {
        const int n = __shfl_up_sync(0xffffffffu, incl, d);
        if (lane >= d) incl += n;
    }
    const unsigned total = (unsigned)__shfl_sync(0xffffffffu, incl, 31);
    unsigned slot = POOL_CAP;
    int refresh = 0;
    if (lane == 0) {
        atomicAdd(&ctrl->hits, 1ull);
        if (total == 0) atomicAdd(&ctrl->false_hits, 1ull);
        else if (ld_relaxed_u32(&ctrl->pool_overflow) == 0u) {
            slot = atomicAdd(&ctrl->count, total);
            if (slot + total > POOL_CAP) atomicExch(&ctrl->pool_overflow, 1u);
            refresh = plan.use_hist && (slot / (unsigned)plan.refresh != (slot + total) / (unsigned)plan.refresh);
        }
    }
    if (total == 0) return;                                      // a false hit of the screen
    slot = __shfl_sync(0xffffffffu, slot, 0);
    refresh = __shfl_sync(0xffffffffu, refresh, 0);
    if (slot >= POOL_CAP) return;                                // the pool is full: the run is void (sticky flag)
    slot += (unsigned)(incl - cnt);
    const long long Wq = ctrl->Wq;
    const int hs = ctrl->hist_shift;
    for (int mid = 0; mid < NMID; ++mid) {
        const int e = v + sC[mid * NLO + lane] + __shfl_sync(0xffffffffu, ux, mid);
        if (mask >> mid & 1u) {
            if (slot < POOL_CAP) {
                Entry en;
                en.key = key_from_i32(e);
                en.q = qs + ((unsigned)mid << LL);
                pool[slot] = en;
                if (plan.use_hist) {
                    const int b = hist_bin(e, Wq, hs);
                    atomicAdd(hist + HIST_COARSE + b, 1u);
                    atomicAdd(hist + (b >> 8), 1u);
                }
            }
            ++slot;
        }
    }
    if (refresh) {
        __threadfence();
        __syncwarp();
        refresh_tau(ctrl, hist, plan, lane);
    }
}

// The persistent kernel. INNER supplies the per-thread tables of the 1024-configuration block and its screen:
//   struct Shared                               instance tables in shared memory
//   struct Regs                                 per-thread tables in registers
//   load_shared(Shared&, tab)                   block-wide copy (followed by __syncthreads in the kernel)
//   init(Regs&, tab, Phi[LOWBITS])              tables of the thread's base state from its ten local fields
//   hit_step(Regs&, Shared&, tab, tauE, Eh, k, sb) -> bool
//                                               "some configuration of the block may have energy <= tauE"; afterwards
//                                               the tables take the Gray step: walk bit k turns on (sb = 1) / off (0)
template <class INNER>
__global__ void __launch_bounds__(WALK_THREADS, 2)
walk_kernel(const Tables* __restrict__ tab, Ctrl* __restrict__ ctrl, Entry* __restrict__ pool,
            unsigned* __restrict__ hist, const __grid_constant__ Plan plan)
{
    __shared__ typename INNER::Shared sh;
    __shared__ int sC[NMID * NLO];
    __shared__ int sDW[1 << LW_MAX];
    __shared__ int sPhiW[LW_MAX][WALK_THREADS];    // per-thread local fields of the walk spins at the base state
    __shared__ int sPhiB[WALK_WARPS][64];          // per-warp local fields of all spins at the unit's first state

    INNER::load_shared(sh, tab);
    for (int i = threadIdx.x; i < NMID * NLO; i += blockDim.x) sC[i] = tab->C[i];
    for (int i = threadIdx.x; i < (1 << LW_MAX); i += blockDim.x) sDW[i] = tab->DW[i];
    __syncthreads();
    if (ctrl->status != 0) return;

    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const int N = plan.N;
    const int* __restrict__ Jq = tab->Jq;

    {
        // ---- take the next unit (ascending q) ----
        unsigned long long u = 0;
        if (lane == 0) u = atomicAdd(&ctrl->next_unit, 1ull);
        u = __shfl_sync(0xffffffffu, u, 0);
        if (u >= plan.total_units) return;
        int s = 0;
        while (s + 1 < plan.nseg && u >= plan.seg[s].first_unit + plan.seg[s].n_units) ++s;
        const int unit_bits = plan.seg[s].unit_bits;
        const unsigned long long qW = plan.seg[s].q0 + ((u - plan.seg[s].first_unit) << unit_bits);
        // ---- ramp-up rule: wait until enough of the earlier states are done (never waits on later units) ----
        const unsigned long long need = plan.seg[s].need_done;
        int dead = 0;
        if (lane == 0) {
            while (ld_relaxed_u64(&ctrl->done_configs) < need) {
                if (ld_relaxed_u32(&ctrl->pool_overflow)) break;
                __nanosleep(100);
            }
            dead = ld_relaxed_u32(&ctrl->pool_overflow) != 0u;
        }
        if (__shfl_sync(0xffffffffu, dead, 0)) return;           // the run is void: stop
        __threadfence();
        unsigned long long tau = ld_relaxed_u64(&ctrl->tau);

        if (unit_bits == LOWBITS) {
            // ---- a2': one block formed exactly, nothing screened (the threshold does not exist yet) ----
            form_block<true>(tab, ctrl, pool, hist, plan, sC, qW, 0, tau, lane);
        } else {
            const int Lw = unit_bits - MIN_CHUNK_BITS;
            const int nlow = LOWBITS + Lw;
            // ---- a2, warp part: Phi_i(qW) for every spin, E(qW) ----
            int plo, phi;
            const int EW = warp_fields(tab, N, qW, lane, plo, phi);
            __syncwarp();
            sPhiB[warp][lane] = plo;
            sPhiB[warp][lane + 32] = phi;
            __syncwarp();
            // ---- a2, lane part: q0 = qW + (lane << nlow) differs from qW in the set lane bits D (spins nlow + j):
            //      Phi_i(q0) = Phi_i(qW) + 2 sum_{a in D} Jq[i][a]
            //      E(q0)     = E(qW) - 2 sum_{a in D} Phi_a(qW) - 4 sum_{a<b in D} Jq[a][b]
            int Phi[LOWBITS];
            int PhiW[LW_MAX];
#pragma unroll
            for (int i = 0; i < LOWBITS; ++i) Phi[i] = sPhiB[warp][i];
#pragma unroll
            for (int i = 0; i < LW_MAX; ++i) PhiW[i] = (i < Lw) ? sPhiB[warp][LOWBITS + i] : 0;
            int Eh = EW;
            for (int j = 0; j < 5 && nlow + j < N; ++j) {
                const bool fl = (lane >> j) & 1;
                const int a = nlow + j;
                const int* col = Jq + a * 64;                    // row a = column a (symmetric): warp-uniform loads
#pragma unroll
                for (int i = 0; i < LOWBITS; ++i) Phi[i] += fl ? 2 * col[i] : 0;
#pragma unroll
                for (int i = 0; i < LW_MAX; ++i) PhiW[i] += (fl && i < Lw) ? 2 * col[LOWBITS + i] : 0;
                int e = -2 * sPhiB[warp][a];
                for (int jj = 0; jj < j; ++jj)
                    if ((lane >> jj) & 1) e -= 4 * col[nlow + jj];
                Eh += fl ? e : 0;
            }
#pragma unroll
            for (int i = 0; i < LW_MAX; ++i) sPhiW[i][threadIdx.x] = PhiW[i];

            typename INNER::Regs R;
            INNER::init(R, tab, Phi);

            const unsigned long long q0_warp = qW;
            int tauE = tau_energy(tau);
            const unsigned nsteps = 1u << Lw;
            for (unsigned t = 0; t < nsteps; ++t) {
                asm volatile("" ::: "memory");             // the tables are re-read every step: keep them out of registers
                // the Gray step that FOLLOWS this block flips walk bit k = ctz(t + 1) (warp-uniform table rows); after
                // the last block of the unit a harmless dummy step is applied
                const unsigned tn = t + 1 < nsteps ? t + 1 : 1u;
                const int k = __ffs(tn) - 1;
                const int sb = ((tn ^ (tn >> 1)) >> k) & 1;
                // ---- a3 + a4: 1024 configurations against the threshold (then the tables move on to step t + 1) ----
                unsigned hits = __ballot_sync(0xffffffffu, INNER::hit_step(R, sh, tab, tauE, Eh, k, sb));
                while (hits) {
                    const int src = __ffs(hits) - 1;
                    hits &= hits - 1;
                    const unsigned gray = t ^ (t >> 1);
                    const unsigned long long qh = q0_warp + ((unsigned long long)src << nlow)
                                                + ((unsigned long long)gray << LOWBITS);
                    const int eh = __shfl_sync(0xffffffffu, Eh, src);
                    form_block<false>(tab, ctrl, pool, hist, plan, sC, qh, eh, tau, lane);
                    tau = ld_relaxed_u64(&ctrl->tau);
                    tauE = tau_energy(tau);
                }
                const int phi_k = sPhiW[k][threadIdx.x];
                Eh += sDW[tn] + (sb ? -2 * phi_k : 2 * phi_k);
                if ((t & 15u) == 15u) {                     // the running S-th best, broadcast from global memory
                    tau = ld_relaxed_u64(&ctrl->tau);
                    tauE = tau_energy(tau);
                }
            }
        }
        // ---- unit complete ----
        __syncwarp();
        if (lane == 0) {
            __threadfence();
            atomicAdd(&ctrl->done_configs, 1ull << unit_bits);
        }
    }
}

}  // namespace ising
