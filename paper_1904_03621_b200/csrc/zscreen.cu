// zscreen.cu -- SURVEY.md section 8 rows a3 + a4 on the 5th-generation tensor cores (tcgen05 / TMEM): the threshold
// screen of a block of 2^14 configurations as ONE dense contraction.
//
// The block energies decompose exactly as in enumerate.cu (the QUBO form of eqs. (2),(3), around the
// thread's base state with the 14 block spins down):
//      E(lo, mid) = Eh - 2 sum_{i in lo} Phi_i - 2 sum_{j in mid} Phi_j + C'(lo, mid),
//      C'(lo, mid) = -4 sum_{a<b both set in lo u mid} Jq_ab        (per instance; lo = spins 0..6, mid = spins 7..13)
// "Does the block hold a configuration with E <= tauE?" is a (min,+) question. Its (+,x) image is the block's
// partition function at inverse temperature lambda (bits per grid unit):
//      Z = sum_{lo,mid} 2^(-lambda (E(lo,mid) - tauE))  >=  2^(-lambda (E_min - tauE)),
// so  E_min <= tauE  implies  Z >= 1, and a block with Z < 1 cannot hold a candidate: THE SCREEN CAN PRODUCE FALSE
// HITS, NEVER A MISS -- provided Z is not under-estimated by more than the margin kept below. Z factorises,
//      Z = 2^L  sum_mid u[mid]  ( sum_lo T[mid][lo] a[lo] ),   T[mid][lo] = 2^(-lambda C'(lo,mid) + t0)   (per instance)
//      a[lo]  = prod_{i in lo}  2^(2 lambda Phi_i) / (largest such product)        in (0, 1]     (per thread and step)
//      u[mid] = prod_{j in mid} 2^(2 lambda Phi_j) / (largest such product)        in (0, 1]
//      L      = lambda (tauE - Eh) - t0 + sum_i max(2 lambda Phi_i, 0)                             (log domain, fp32)
// and the inner sum over lo is a GEMM: D[thread][mid] = sum_lo A[thread][lo] T[mid][lo] with A = the a-vectors of the
// 128 threads of the CTA -- M = 128 (threads), N = 128 (mid), K = 128 (lo), bf16 inputs, fp32 accumulation in TMEM,
// 2 flop per configuration. Per step a thread generates its A row (190 multiplies -- the last level in packed bf16 --
// written in the UMMA canonical layout), one elected thread issues 8 tcgen05.mma (K = 16 each), and every thread folds
// its own D row (tcgen05.ld) with the u factors in radix 4: 180 multiply-adds for 2^14 configurations, against 2^13
// packed add-mins in enumerate16.cu. A flagged block is formed exactly (int32) by the warp, 16 x 1024 configurations
// (push_block below: the ALU kernels' form_block again), so what reaches the pool is identical to the other kernels.
//
// Why the screen is rigorous (DESIGN.md section 6b has the full argument):
//   * all terms are positive, so rounding only perturbs Z relatively: bf16 keeps 8 significant bits, so one rounding
//     to nearest is off by at most 2^-8 relative. T is rounded to bf16 once, an entry of a three times (the partial
//     product of five spins, the factor of the other two, their bf16 product): FOUR bf16 roundings per term,
//     -4 log2(1 - 2^-8) = 0.0226 bits. The fp32 products inside the tensor core are exact; accumulation, the u-fold
//     and the factor chain add < 2^-11 relative (0.0008 bits); L -- one fp32 multiply-add of an EXACT integer,
//     L = lambda (tauE - Eh + 2 sum_i max(Phi_i, 0)) - t0 -- is good to 2^-22 |L| < 1e-4 bits wherever the test can go
//     either way (|L| < 200). Total < 0.024 bits. The test flags a block unless  log2(Z~) + L < -Z_MARGIN = -0.05 ;
//   * underflow: a term of a configuration with E <= tauE has  log2 a + log2 T + log2 u >= -L; with |log2 T| <= THETA
//     (lambda is chosen from the range of C') none of its partial products is below 2^-(L + THETA), so for
//     L <= L_SAFE = 126 - THETA - 8 it cannot underflow; blocks with L > L_SAFE are flagged unconditionally
//     (their crude bound is far below tauE: they almost always do hold a candidate);
//   * overflow cannot happen (a, u <= 1, T <= 2^THETA), and a NaN can only make the comparison fail, i.e. flag.
#include <cuda_bf16.h>

#include "walk.cuh"

namespace ising {

constexpr int Z_THREADS = 128;
constexpr unsigned Z_LBO = 128, Z_SBO = 2048;          // UMMA canonical K-major layout without swizzle (bytes)
constexpr float Z_THETA = 40.f;                        // half range of log2 T
constexpr float Z_L_SAFE = 126.f - Z_THETA - 8.f;
// Margin of the screen in bits. The error budget is 0.024 bits, of which 0.0226 are the Z_BF16_ROUNDINGS roundings to
// bf16 (2^-8 each) a term goes through (file header): a change of the row generation that adds a bf16
// rounding must revisit this constant.
constexpr int Z_BF16_ROUNDINGS = 4;
constexpr float Z_MARGIN = 0.05f;
static_assert(Z_BF16_ROUNDINGS * 0.005647 + 0.0015 < Z_MARGIN * 0.5 + 0.0, "margin: at least twice the error budget (-log2(1 - 2^-8) = 0.005647 bits per bf16 rounding)");
// kind::f16 instruction descriptor: D fp32, A and B bf16, both K-major, N = 128, M = 128
constexpr unsigned Z_IDESC = (1u << 4) | (1u << 7) | (1u << 10) | ((unsigned)(128 >> 3) << 17) | ((unsigned)(128 >> 4) << 24);
constexpr int Z_SMEM_BYTES = 32768 + 32768;            // T table + A tile (dynamic shared memory)

__device__ __forceinline__ unsigned smem_u32(const void* p) { return (unsigned)__cvta_generic_to_shared(p); }

__device__ __forceinline__ unsigned long long umma_desc(unsigned saddr)
{
    return (unsigned long long)((saddr >> 4) & 0x3fffu) | ((unsigned long long)(Z_LBO >> 4) << 16) |
           ((unsigned long long)(Z_SBO >> 4) << 32) | (1ull << 46);         // version 1, no swizzle, base offset 0
}

__device__ __forceinline__ float ex2f(float x) { float r; asm("ex2.approx.ftz.f32 %0, %1;" : "=f"(r) : "f"(x)); return r; }
__device__ __forceinline__ float lg2f(float x) { float r; asm("lg2.approx.ftz.f32 %0, %1;" : "=f"(r) : "f"(x)); return r; }
// packed fp32 pairs (FMUL2 / FFMA2): two lanes per issue slot
__device__ __forceinline__ unsigned long long pk2(float lo, float hi) { unsigned long long r; asm("mov.b64 %0, {%1, %2};" : "=l"(r) : "f"(lo), "f"(hi)); return r; }
__device__ __forceinline__ void upk2(unsigned long long v, float& lo, float& hi) { asm("mov.b64 {%0, %1}, %2;" : "=f"(lo), "=f"(hi) : "l"(v)); }
__device__ __forceinline__ unsigned long long mul2(unsigned long long a, unsigned long long b) { unsigned long long r; asm("mul.rn.f32x2 %0, %1, %2;" : "=l"(r) : "l"(a), "l"(b)); return r; }
__device__ __forceinline__ unsigned long long fma2(unsigned long long a, unsigned long long b, unsigned long long c) { unsigned long long r; asm("fma.rn.f32x2 %0, %1, %2, %3;" : "=l"(r) : "l"(a), "l"(b), "l"(c)); return r; }
__device__ __forceinline__ unsigned hmul2_bf16(unsigned a, unsigned b) { unsigned r; asm("mul.rn.bf16x2 %0, %1, %2;" : "=r"(r) : "r"(a), "r"(b)); return r; }
__device__ __forceinline__ unsigned pack_bf16(float lo, float hi)
{
    unsigned r;
    asm("cvt.rn.bf16x2.f32 %0, %1, %2;" : "=r"(r) : "f"(hi), "f"(lo));     // d.hi = first source, d.lo = second
    return r;
}

// ---- per-instance tables of the screen: one block, after stage_kernel ----
__global__ void __launch_bounds__(1024) ztables_kernel(const Tables* __restrict__ tab, const Ctrl* __restrict__ ctrl,
                                                       ZTables* __restrict__ zt, int N)
{
    if (ctrl->status != 0) return;
    __shared__ int s_min, s_max;
    __shared__ float s_lambda, s_t0;
    const int tid = threadIdx.x;
    const int* __restrict__ Jq = tab->Jq;
    if (tid == 0) { s_min = 0x7fffffff; s_max = -0x7fffffff; }
    __syncthreads();
    int mn = 0x7fffffff, mx = -0x7fffffff;
    for (int x = tid; x < (1 << ZB); x += blockDim.x) {
        int acc = 0;
        for (int a = 0; a < ZB; ++a)
            if (x >> a & 1)
                for (int b = a + 1; b < ZB; ++b)
                    if (x >> b & 1) acc += Jq[a * 64 + b];              // rows/columns >= N are zero
        const int c = -4 * acc;
        zt->Cz[x] = c;
        mn = min(mn, c);
        mx = max(mx, c);
    }
    atomicMin(&s_min, mn);
    atomicMax(&s_max, mx);
    for (int idx = tid; idx < LW_MAX * 16; idx += blockDim.x) {
        const int k = idx >> 4, i = idx & 15;
        zt->DPhi[idx] = (i < ZB && ZB + k < 64) ? 2 * Jq[i * 64 + ZB + k] : 0;
    }
    for (int t = tid; t < (1 << LW_MAX); t += blockDim.x) {
        int v = 0;
        if (t > 0) {
            const int k = __ffs(t) - 1;
            const int gnew = t ^ (t >> 1);
            const int sgn = (gnew >> k & 1) ? 1 : -1;
            const int R = gnew & ~(1 << k);
            int acc = 0;
            for (int j = 0; j < LW_MAX; ++j)
                if ((R >> j & 1) && ZB + k < 64 && ZB + j < 64) acc += Jq[(ZB + k) * 64 + ZB + j];
            v = -sgn * 4 * acc;
        }
        zt->DWz[t] = v;
    }
    __syncthreads();
    if (tid == 0) {
        // lambda: the table spans 2 THETA bits; an instance without couplings inside the block gets a sharp screen
        const double range = (double)s_max - (double)s_min;
        double lam = range > 0.0 ? 2.0 * (double)Z_THETA / range : 16.0;
        if (lam > 16.0) lam = 16.0;
        s_lambda = (float)lam;
        s_t0 = (float)(lam * 0.5 * ((double)s_max + (double)s_min));
        zt->lambda = s_lambda;
        zt->t0 = s_t0;
        zt->cmin = s_min;
        zt->cmax = s_max;
    }
    __syncthreads();
    const double lam = (double)s_lambda, t0 = (double)s_t0;
    unsigned short* Tb = reinterpret_cast<unsigned short*>(zt->Tb);
    for (int x = tid; x < (1 << ZB); x += blockDim.x) {
        const int lo = x & 127, mid = x >> 7;
        const double e = -lam * (double)zt->Cz[x] + t0;                  // |e| <= THETA (+ rounding of lambda, t0)
        const __nv_bfloat16 v = __float2bfloat16_rn((float)exp2(e));
        // canonical layout of the B operand: row = mid (N index), column = lo (K index)
        const unsigned off = (unsigned)(mid >> 3) * Z_SBO + (unsigned)(lo >> 3) * Z_LBO + (unsigned)(mid & 7) * 16u + (unsigned)(lo & 7) * 2u;
        Tb[off >> 1] = __bfloat16_as_ushort(v);
    }
}

// a4, second half: the whole warp forms the 1024 energies of one block exactly (int32 grid units) and pushes the
// survivors. qh = the block's state with lo and mid bits zero, eh = its grid energy; lane l holds the block's tables
// vx = V[lo = l], ux = U[mid = l] (common.cuh vocabulary). Two passes: mark the survivors, reserve their pool slots with
// ONE atomic per block, then write. Returns the number of survivors. (walk.cuh form_block is the ALU kernels' version of
// the same steps; this one counts the hit statistics in registers -- every global round trip of a flagged block is paid
// by a whole CTA -- reads the plan's fields once, and updates the histogram once per bin and warp. It is kept apart so
// that the register allocation of the ALU kernels' loop, which ptxas ties to the code of the function it calls, stays
// the conflict-free one: enumerate16.cu header.)
__device__ __forceinline__ unsigned push_block(Ctrl* __restrict__ ctrl, Entry* __restrict__ pool, unsigned* __restrict__ hist,
                                           const Plan& plan, const int* sC, unsigned long long qh, int vx, int ux, int eh,
                                           unsigned long long tau, int lane)
{
    const int tauE = tau_energy(tau);
    const unsigned qc = tau_qc(tau);
    const unsigned long long tauQ = qc == QC_NONE ? Q_MAX : plan.q_begin + ((unsigned long long)qc << plan.qshift);
    // (the plan is reached through a reference here: read its fields once, not inside the loops)
    const int loE = plan.loE, use_hist = plan.use_hist;
    const unsigned long long q_end = plan.q_end;
    const unsigned refresh_every = (unsigned)plan.refresh;
    const unsigned long long qs = qh + (unsigned)lane;
    const int v = vx + eh;
    unsigned mask = 0;
#pragma unroll 8
    for (int mid = 0; mid < NMID; ++mid) {
        const int e = v + sC[mid * NLO + lane] + __shfl_sync(0xffffffffu, ux, mid);
        const unsigned long long q = qs + ((unsigned)mid << LL);
        const bool pass = (e < tauE || (e == tauE && q < tauQ)) && e >= loE && q < q_end;
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
        if (total != 0 && ld_relaxed_u32(&ctrl->pool_overflow) == 0u) {
            slot = atomicAdd(&ctrl->count, total);
            if (slot + total > POOL_CAP) atomicExch(&ctrl->pool_overflow, 1u);
            refresh = use_hist && (slot / refresh_every != (slot + total) / refresh_every);
        }
    }
    if (total == 0) return 0u;                                   // a false hit of the screen
    slot = __shfl_sync(0xffffffffu, slot, 0);
    refresh = __shfl_sync(0xffffffffu, refresh, 0);
    if (slot >= POOL_CAP) return total;                          // the pool is full: the run is void (sticky flag)
    slot += (unsigned)(incl - cnt);
    const long long Wq = ctrl->Wq;
    const int hs = ctrl->hist_shift;
    for (int mid = 0; mid < NMID; ++mid) {
        const int e = v + sC[mid * NLO + lane] + __shfl_sync(0xffffffffu, ux, mid);
        const bool mine = (mask >> mid & 1u) != 0u;
        const unsigned act = __ballot_sync(0xffffffffu, mine);
        if (mine) {
            if (slot < POOL_CAP) {
                Entry en;
                en.key = key_from_i32(e);
                en.q = qs + ((unsigned)mid << LL);
                pool[slot] = en;
            }
            ++slot;
            if (use_hist) {
                // lanes of one bin count together: on degenerate instances (a few dozen distinct energies) thousands of
                // candidates of the threshold-free first blocks would otherwise queue on the same two counters
                const int b = hist_bin(e, Wq, hs);
                const unsigned peers = __match_any_sync(act, b);
                if ((unsigned)lane == (unsigned)(__ffs(peers) - 1)) {
                    const unsigned n = (unsigned)__popc(peers);
                    atomicAdd(hist + HIST_COARSE + b, n);
                    atomicAdd(hist + (b >> 8), n);
                }
            }
        }
    }
    if (refresh) {
        __threadfence();
        __syncwarp();
        refresh_tau(ctrl, hist, plan, lane);
    }
    return total;
}

// ---- a flagged block of 2^14 configurations, formed exactly by the warp: sixteen blocks of 1024 (push_block above).
// P = the fourteen local fields of the flagged thread at the block's base state (block spins down), e0 = its grid
// energy, both already broadcast to every lane. Setting block spin 10 + a raises the field of spin i by 2 Jq[i][10 + a],
// so the lane's tables of the ten low spins and the base energy of sub-block `sub` follow from those of sub-block 0 by at
// most four additions each (eqs. (2),(3)):
//      E(q0 u A) = E(q0) - 2 sum_{a in A} Phi_a(q0) - 4 sum_{a<b in A} Jq_ab .
// (Forming each sub-block from scratch -- every field re-summed over all N spins -- cost 75 us per flagged block, during
// which the other three warps of the CTA wait at the step barrier: the tail of every launch of a few steps per CTA.) ----
// Returns the number of sub-blocks that held a candidate; the threshold is re-read after those only.
static __device__ __forceinline__ unsigned form_flagged(const Tables* __restrict__ tab, Ctrl* __restrict__ ctrl,
                                                     Entry* __restrict__ pool, unsigned* __restrict__ hist, const Plan& plan,
                                                     const int* sC, const int (&Pin)[ZB], int e0, unsigned long long qh,
                                                     unsigned long long& tau_io, int lane)
{
    static_assert(ZB == LOWBITS + 4, "sixteen sub-blocks");
    const int* __restrict__ Jq = tab->Jq;
    // reference arguments of an out-of-line function live in local memory, and with no L1 left on the SM every access
    // to it is an L2 round trip: read them once, keep registers
    int P[ZB];
#pragma unroll
    for (int i = 0; i < ZB; ++i) P[i] = Pin[i];
    unsigned long long tau = tau_io;
    int vx0 = tab->QL[lane], ux0 = tab->QM[lane];
#pragma unroll
    for (int i = 0; i < LL; ++i) {
        if (lane >> i & 1) { vx0 -= 2 * P[i]; ux0 -= 2 * P[LL + i]; }
    }
    int dvx[4], dux[4];
#pragma unroll
    for (int a = 0; a < 4; ++a) {
        int sv = 0, su = 0;
#pragma unroll
        for (int i = 0; i < LL; ++i) {
            if (lane >> i & 1) { sv += Jq[i * 64 + LOWBITS + a]; su += Jq[(LL + i) * 64 + LOWBITS + a]; }
        }
        dvx[a] = -4 * sv;
        dux[a] = -4 * su;
    }
    int jp[4][4];                                           // couplings among the four upper block spins (read once: L2)
#pragma unroll
    for (int a = 0; a < 4; ++a)
#pragma unroll
        for (int b = 0; b < a; ++b) jp[b][a] = 4 * Jq[(LOWBITS + b) * 64 + LOWBITS + a];
    unsigned n_true = 0;
#pragma unroll 1
    for (int sub = 0; sub < 16; ++sub) {
        int vx = vx0, ux = ux0, eh = e0;
#pragma unroll
        for (int a = 0; a < 4; ++a) {
            if (sub >> a & 1) {
                vx += dvx[a];
                ux += dux[a];
                eh -= 2 * P[LOWBITS + a];
#pragma unroll
                for (int b = 0; b < a; ++b)
                    if (sub >> b & 1) eh -= jp[b][a];
            }
        }
        if (push_block(ctrl, pool, hist, plan, sC, qh + ((unsigned long long)sub << LOWBITS), vx, ux, eh, tau, lane)) {
            ++n_true;
            tau = ld_relaxed_u64(&ctrl->tau);
        }
    }
    tau_io = tau;
    return n_true;
}

// ---- all flagged blocks of one warp and step. myC: 4 KB of shared memory for the C table of the 1024-configuration
// blocks -- with three CTAs of 75 KB the SM has no L1 left, and every one of the 16 x 32 table reads of a flagged block
// would be an L2 round trip (measured: 70 000 clocks per flagged block, the whole CTA waiting); the warp's own eight row
// groups of the A tile (8 KB, contiguous in the canonical layout) are free here: the MMAs of this step are complete and
// only this warp writes these rows again, in the next row generation. Phi has already taken the Gray step that follows
// this block (row dphi of the step table, direction sb): the fields of THIS step are recovered first. ----
static __device__ __noinline__ unsigned handle_flagged(const Tables* __restrict__ tab, Ctrl* __restrict__ ctrl,
                                                       Entry* __restrict__ pool, unsigned* __restrict__ hist, const Plan& plan,
                                                       int* myC, const int* dphi, int sb, const int (&PhiNext)[ZB], int Eh,
                                                       unsigned hits, unsigned long long q_step, int nlow,
                                                       unsigned long long& tau_io, int lane)
{
    {
        const int4* __restrict__ src4 = reinterpret_cast<const int4*>(tab->C);
#pragma unroll
        for (int i = 0; i < (NMID * NLO / 4) / 32; ++i) reinterpret_cast<int4*>(myC)[i * 32 + lane] = src4[i * 32 + lane];
        __syncwarp();
    }
    int Pt[ZB];
#pragma unroll
    for (int i = 0; i < ZB; ++i) Pt[i] = PhiNext[i] - (sb ? dphi[i] : -dphi[i]);
    unsigned long long tau = tau_io;
    unsigned n_true = 0;
    while (hits) {
        const int src = __ffs(hits) - 1;
        hits &= hits - 1;
        int P[ZB];
#pragma unroll
        for (int i = 0; i < ZB; ++i) P[i] = __shfl_sync(0xffffffffu, Pt[i], src);
        const int e0 = __shfl_sync(0xffffffffu, Eh, src);
        n_true += form_flagged(tab, ctrl, pool, hist, plan, myC, P, e0, q_step + ((unsigned long long)src << nlow), tau, lane);
    }
    tau_io = tau;
    return n_true;
}

// ---- the screen kernel: one CTA of 128 threads per unit of 2^(21 + Lw) configurations ----
__global__ void __launch_bounds__(Z_THREADS, 3)
zwalk_kernel(const Tables* __restrict__ tab, const ZTables* __restrict__ zt, Ctrl* __restrict__ ctrl,
             Entry* __restrict__ pool, unsigned* __restrict__ hist, const __grid_constant__ Plan plan)
{
    extern __shared__ __align__(1024) unsigned char zsmem[];
    unsigned char* sT = zsmem;                       // 32 KB: B operand (the instance table)
    unsigned char* sA = zsmem + 32768;               // 32 KB: A operand (one row per thread)
    __shared__ __align__(8) unsigned long long mbar[1];
    __shared__ unsigned s_tmem;
    __shared__ unsigned long long s_unit;
    __shared__ int sDWz[1 << LW_MAX];
    __shared__ __align__(16) int sDPhi[LW_MAX * 16];
    __shared__ int sPhiW[LW_MAX][Z_THREADS];
    int (*sPhiB)[64] = reinterpret_cast<int (*)[64]>(sA);   // base-state scratch: lives in the A tile until the first step

    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    if (ctrl->status != 0) return;
    // ---- take a unit ----
    if (tid == 0) s_unit = atomicAdd(&ctrl->next_unit, 1ull);
    for (int i = tid; i < 2048; i += Z_THREADS) reinterpret_cast<uint4*>(sT)[i] = zt->Tb[i];
    for (int i = tid; i < (1 << LW_MAX); i += Z_THREADS) sDWz[i] = zt->DWz[i];
    for (int i = tid; i < LW_MAX * 16; i += Z_THREADS) sDPhi[i] = zt->DPhi[i];
    if (tid == 0) {
        asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" :: "r"(smem_u32(&mbar[0])), "r"(1));
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    __syncthreads();
    const unsigned long long u = s_unit;
    if (u >= plan.total_units) return;
    int s = 0;
    while (s + 1 < plan.nseg && u >= plan.seg[s].first_unit + plan.seg[s].n_units) ++s;
    const int unit_bits = plan.seg[s].unit_bits;
    const int Lw = unit_bits - (ZB + 7);
    const int nlow = ZB + Lw;
    const unsigned long long qU = plan.seg[s].q0 + ((u - plan.seg[s].first_unit) << unit_bits);
    if (tid == 0) {
        const unsigned long long need = plan.seg[s].need_done;
        while (ld_relaxed_u64(&ctrl->done_configs) < need) {
            if (ld_relaxed_u32(&ctrl->pool_overflow)) break;
            __nanosleep(100);
        }
    }
    __syncwarp();
    if (warp == 0) {
        asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], %1;" :: "r"(smem_u32(&s_tmem)), "r"(128));
        asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;");
    }
    asm volatile("fence.proxy.async.shared::cta;" ::: "memory");          // the table copy is read by the tensor core
    asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory");
    __syncthreads();
    asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
    const unsigned tmem = s_tmem;
    const bool dead = ld_relaxed_u32(&ctrl->pool_overflow) != 0u;         // the run is void: only release TMEM

    const int N = plan.N;
    const int* __restrict__ Jq = tab->Jq;
    const float lambda = zt->lambda, t0 = zt->t0;
    unsigned long long flagged = 0ull;
    unsigned sub_true = 0;                                  // exactly formed blocks of 1024 that held a candidate

    if (!dead) {
        // ---- a2: base state. Warp: Phi_i(qW), E(qW) for the warp's first state; lane: its 5 lane bits on top ----
        const unsigned long long qW = qU + ((unsigned long long)warp << (nlow + 5));
        int plo, phi;
        const int EW = warp_fields(tab, N, qW, lane, plo, phi);
        sPhiB[warp][lane] = plo;
        sPhiB[warp][lane + 32] = phi;
        __syncwarp();
        int Phi[ZB];
        int PhiW[LW_MAX];
#pragma unroll
        for (int i = 0; i < ZB; ++i) Phi[i] = sPhiB[warp][i];
#pragma unroll
        for (int i = 0; i < LW_MAX; ++i) PhiW[i] = (i < Lw) ? sPhiB[warp][ZB + i] : 0;
        int Eh = EW;
        for (int j = 0; j < 5 && nlow + j < N; ++j) {
            const bool fl = (lane >> j) & 1;
            const int a = nlow + j;
            const int* col = Jq + a * 64;
#pragma unroll
            for (int i = 0; i < ZB; ++i) Phi[i] += fl ? 2 * col[i] : 0;
#pragma unroll
            for (int i = 0; i < LW_MAX; ++i) PhiW[i] += (fl && i < Lw) ? 2 * col[ZB + i] : 0;
            int e = -2 * sPhiB[warp][a];
            for (int jj = 0; jj < j; ++jj)
                if ((lane >> jj) & 1) e -= 4 * col[nlow + jj];
            Eh += fl ? e : 0;
        }
#pragma unroll
        for (int i = 0; i < LW_MAX; ++i) sPhiW[i][tid] = PhiW[i];
        __syncthreads();                                 // the scratch in the A tile is dead from here on

        unsigned long long tau = ld_relaxed_u64(&ctrl->tau);
        int tauE = tau_energy(tau);
        const float two_lambda = 2.f * lambda;
        const unsigned rowoff = (unsigned)(tid >> 3) * Z_SBO + (unsigned)(tid & 7) * 16u;
        const unsigned nsteps = 1u << Lw;

        // Factors of one step from the fourteen local fields, and the thread's A row into buffer `buf`:
        //   bit set multiplies the weight by 2^y, y = 2 lambda Phi; normalised so that the larger of the two factors of
        //   a spin is exactly 1. a[lo] = product over the 7 lo spins, 128 values, bf16, canonical layout; products in
        //   packed fp32 pairs (FMUL2): pair p of Q holds lo = 2p (low lane: spin 0 down) and 2p + 1 (spin 0 up).
        // Returns the mid-spin factors (for the fold). The log-domain offset L is formed from EXACT integers,
        // L = lambda (tauE - Eh + 2 sum_i max(Phi_i, 0)) - t0 (spos below), so that its error is RELATIVE (2^-23 |L|)
        // however large the fields are in grid units (summing the fp32 terms lambda (tauE - Eh) and 2 lambda Phi_i
        // separately would cancel catastrophically on instances with strong fields and weak couplings in the block).
        auto gen_row = [&](int buf, const int (&Ph)[ZB], float (&m0)[7], float (&m1)[7]) {
            float r0[ZB], r1[ZB];
#pragma unroll
            for (int i = 0; i < ZB; ++i) {
                const float y = two_lambda * (float)Ph[i];
                const float e = ex2f(-fabsf(y));
                r1[i] = y >= 0.f ? 1.f : e;
                r0[i] = y >= 0.f ? e : 1.f;
            }
#pragma unroll
            for (int i = 0; i < 7; ++i) { m0[i] = r0[7 + i]; m1[i] = r1[7 + i]; }
            unsigned long long Q[16];
            Q[0] = pk2(r0[0], r1[0]);
#pragma unroll
            for (int b = 1; b < 5; ++b) {
                const unsigned long long f0 = pk2(r0[b], r0[b]), f1 = pk2(r1[b], r1[b]);
#pragma unroll
                for (int j = (1 << (b - 1)) - 1; j >= 0; --j) {
                    const unsigned long long v = Q[j];
                    Q[j + (1 << (b - 1))] = mul2(v, f1);
                    Q[j] = mul2(v, f0);
                }
            }
            unsigned char* myrow = sA + (unsigned)buf * 32768u + rowoff;
            // the last two lo spins in packed bf16 (HMUL2.BF16): the 32 partial products and the four factor products are
            // rounded to bf16 once each and multiplied in bf16 -- three roundings per element instead of one, budgeted in
            // the margin -- which saves the 64 fp32 -> bf16 conversions of the row
            unsigned Qb[16];
#pragma unroll
            for (int p = 0; p < 16; ++p) { float lo, hi; upk2(Q[p], lo, hi); Qb[p] = pack_bf16(lo, hi); }
#pragma unroll
            for (int c = 0; c < 4; ++c) {
                const float f = ((c & 1) ? r1[5] : r0[5]) * ((c & 2) ? r1[6] : r0[6]);
                const unsigned Fb = pack_bf16(f, f);
#pragma unroll
                for (int g = 0; g < 4; ++g) {
                    uint4 w;
                    w.x = hmul2_bf16(Qb[4 * g + 0], Fb);
                    w.y = hmul2_bf16(Qb[4 * g + 1], Fb);
                    w.z = hmul2_bf16(Qb[4 * g + 2], Fb);
                    w.w = hmul2_bf16(Qb[4 * g + 3], Fb);
                    *reinterpret_cast<uint4*>(myrow + (unsigned)(4 * c + g) * Z_LBO) = w;   // k-chunk lo/8 = 4c + g
                }
            }
            asm volatile("fence.proxy.async.shared::cta;" ::: "memory");    // the row is read by the tensor core
        };
        // One elected thread: D[buf] = A[buf] x T^T, eight K = 16 slices, completion signalled on mbar[buf]. The two base
        // descriptors are formed once (rebuilt per MMA they are a chain of ~17 uniform-datapath instructions each).
        const unsigned long long desc_a0 = umma_desc(smem_u32(sA)), desc_b0 = umma_desc(smem_u32(sT));
        auto issue_mma = [&](int buf) {
            asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
#pragma unroll
            for (int ks = 0; ks < 8; ++ks) {
                // K slice ks starts 2 LBO bytes further on: + 16 in the descriptors' 16-byte address field (no carry out
                // of its 14 bits: shared memory ends below 256 KB)
                const unsigned long long da = desc_a0 + (unsigned long long)(ks * (2 * Z_LBO >> 4));
                const unsigned long long db = desc_b0 + (unsigned long long)(ks * (2 * Z_LBO >> 4));
                const unsigned acc = ks > 0 ? 1u : 0u;
                asm volatile("{\n\t.reg .pred p;\n\tsetp.ne.b32 p, %4, 0;\n\t"
                             "tcgen05.mma.cta_group::1.kind::f16 [%0], %1, %2, %3, p;\n\t}"
                             :: "r"(tmem + (unsigned)buf * 128u), "l"(da), "l"(db), "r"(Z_IDESC), "r"(acc) : "memory");
            }
            asm volatile("tcgen05.commit.cta_group::1.mbarrier::arrive::one.shared::cluster.b64 [%0];"
                         :: "r"(smem_u32(&mbar[buf])) : "memory");
        };

        // ---- one step: rows -> tensor core -> fold. Three CTAs share an SM (single A tile, single accumulator), so
        //      the phases of one CTA overlap with the other two. (A software pipeline inside the CTA -- two A tiles,
        //      two accumulators -- was measured and dropped: the larger footprint leaves two CTAs per SM, and with eight
        //      warps per SM the dependent chains of the row generation and the fold are not hidden: 4.2e14 against
        //      4.9e14 configurations/s.) ----
        float m0[7], m1[7];
        for (unsigned t = 0; t < nsteps; ++t) {
            int spos = 0;                                   // sum_i max(Phi_i, 0) of THIS step's fields
#pragma unroll
            for (int i = 0; i < ZB; ++i) spos += max(Phi[i], 0);
            // (a threshold read a moment ago is never tighter than the current one: conservative)
            const float Lp = fmaf(lambda, (float)(tauE - Eh + 2 * spos), -t0);      // |integer| < 2^31 (4 Wq + 2^30)
            gen_row(0, Phi, m0, m1);
            asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory");
            __syncthreads();       // every A row is written; every TMEM read of the previous step is done
            if (tid == 0) issue_mma(0);
            // ---- while the tensor core works: the Gray step that follows this block (walk bit k = ctz(t + 1)) ----
            const unsigned tn = t + 1 < nsteps ? t + 1 : 1u;
            const int k = __ffs(tn) - 1;
            const int sb = ((tn ^ (tn >> 1)) >> k) & 1;
            const int EhNext = Eh + sDWz[tn] + (sb ? -2 : 2) * sPhiW[k][tid];
            {
                const int4* dp = reinterpret_cast<const int4*>(sDPhi + k * 16);
#pragma unroll
                for (int x = 0; x < 4; ++x) {
                    const int4 d = dp[x];
                    if (4 * x + 0 < ZB) Phi[4 * x + 0] += sb ? d.x : -d.x;
                    if (4 * x + 1 < ZB) Phi[4 * x + 1] += sb ? d.y : -d.y;
                    if (4 * x + 2 < ZB) Phi[4 * x + 2] += sb ? d.z : -d.z;
                    if (4 * x + 3 < ZB) Phi[4 * x + 3] += sb ? d.w : -d.w;
                }
            }
            // ---- wait for the accumulator, fold this thread's row: R = sum_mid u[mid] D[mid] ----
            asm volatile("{\n\t.reg .pred P1;\n\tZWAIT_%=:\n\t"
                         "mbarrier.try_wait.parity.shared::cta.b64 P1, [%0], %1;\n\t"
                         "@P1 bra ZDONE_%=;\n\tbra ZWAIT_%=;\n\tZDONE_%=:\n\t}"
                         :: "r"(smem_u32(&mbar[0])), "r"(t & 1u) : "memory");
            __syncwarp();
            asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
            // the fold in packed pairs (FMUL2 / FFMA2): the stages of mid bits 1..6 combine whole pairs (columns 2p, 2p+1);
            // mid bit 0 (spin 7), which sits inside a pair, comes last. All four loads are issued before the one wait so
            // that the four chunk folds are independent chains.
            unsigned v[4][32];
#pragma unroll
            for (int c = 0; c < 4; ++c) {
                const unsigned taddr = tmem + ((unsigned)(warp * 32) << 16) + (unsigned)(c * 32);
                asm volatile("tcgen05.ld.sync.aligned.32x32b.x32.b32 "
                             "{%0, %1, %2, %3, %4, %5, %6, %7, %8, %9, %10, %11, %12, %13, %14, %15, "
                             "%16, %17, %18, %19, %20, %21, %22, %23, %24, %25, %26, %27, %28, %29, %30, %31}, [%32];"
                             : "=r"(v[c][0]), "=r"(v[c][1]), "=r"(v[c][2]), "=r"(v[c][3]), "=r"(v[c][4]), "=r"(v[c][5]), "=r"(v[c][6]), "=r"(v[c][7]),
                               "=r"(v[c][8]), "=r"(v[c][9]), "=r"(v[c][10]), "=r"(v[c][11]), "=r"(v[c][12]), "=r"(v[c][13]), "=r"(v[c][14]), "=r"(v[c][15]),
                               "=r"(v[c][16]), "=r"(v[c][17]), "=r"(v[c][18]), "=r"(v[c][19]), "=r"(v[c][20]), "=r"(v[c][21]), "=r"(v[c][22]), "=r"(v[c][23]),
                               "=r"(v[c][24]), "=r"(v[c][25]), "=r"(v[c][26]), "=r"(v[c][27]), "=r"(v[c][28]), "=r"(v[c][29]), "=r"(v[c][30]), "=r"(v[c][31])
                             : "r"(taddr) : "memory");
            }
            asm volatile("tcgen05.wait::ld.sync.aligned;" ::: "memory");
            // Radix 4: two mid bits per stage, out = sum_{ab} x_ab (g_a g'_b) -- one multiply and three multiply-adds per
            // output with four coefficient products formed once per step, instead of six operations in two radix-2
            // stages: 84 packed operations per row instead of 126 (the coefficients are scalars broadcast to both lanes).
            unsigned long long part[4];
            unsigned long long cA[4], cB[4], cC[4];
#pragma unroll
            for (int ab = 0; ab < 4; ++ab) {
                const float fa = ((ab & 1) ? m1[1] : m0[1]) * ((ab & 2) ? m1[2] : m0[2]);     // mid bits 1, 2 = spins 8, 9
                const float fb = ((ab & 1) ? m1[3] : m0[3]) * ((ab & 2) ? m1[4] : m0[4]);     // mid bits 3, 4 = spins 10, 11
                const float fc = ((ab & 1) ? m1[5] : m0[5]) * ((ab & 2) ? m1[6] : m0[6]);     // mid bits 5, 6 = spins 12, 13
                cA[ab] = pk2(fa, fa); cB[ab] = pk2(fb, fb); cC[ab] = pk2(fc, fc);
            }
#pragma unroll
            for (int c = 0; c < 4; ++c) {
                // pair p covers mid = 32 c + 2p, 2p + 1; bit b of mid is bit b - 1 of p
                unsigned long long y[4];
#pragma unroll
                for (int g = 0; g < 4; ++g) {
                    unsigned long long x[4];
#pragma unroll
                    for (int j = 0; j < 4; ++j)
                        x[j] = pk2(__uint_as_float(v[c][2 * (4 * g + j)]), __uint_as_float(v[c][2 * (4 * g + j) + 1]));
                    y[g] = fma2(x[3], cA[3], fma2(x[2], cA[2], fma2(x[1], cA[1], mul2(x[0], cA[0]))));
                }
                part[c] = fma2(y[3], cB[3], fma2(y[2], cB[2], fma2(y[1], cB[1], mul2(y[0], cB[0]))));
            }
            // mid bits 5, 6 select the chunk; mid bit 0 = spin 7 sits inside the pair and comes last
            const unsigned long long hh = fma2(part[3], cC[3], fma2(part[2], cC[2], fma2(part[1], cC[1], mul2(part[0], cC[0]))));
            float Rlo, Rhi;
            upk2(hh, Rlo, Rhi);
            const float R = fmaf(Rhi, m1[0], Rlo * m0[0]);
            // ---- a4: flag unless the block provably holds no configuration with E <= tauE ----
            const bool clear = (lg2f(R) + Lp < -Z_MARGIN) && (Lp <= Z_L_SAFE);
            unsigned hits = __ballot_sync(0xffffffffu, !clear);
            flagged += __popc(hits);
            if (hits) {
                // (out of line: the registers of this rare path must not weigh on the loop; the arguments that go by
                // reference are COPIES made here, so that Phi and tau themselves never have their address taken --
                // otherwise they live in local memory and every step pays their stores)
                int phi_copy[ZB];
#pragma unroll
                for (int i = 0; i < ZB; ++i) phi_copy[i] = Phi[i];
                unsigned long long tau_copy = tau;
                sub_true += handle_flagged(tab, ctrl, pool, hist, plan, reinterpret_cast<int*>(sA + (unsigned)warp * 8192u),
                                           sDPhi + k * 16, sb, phi_copy, Eh, hits,
                                           qW + ((unsigned long long)(t ^ (t >> 1)) << ZB), nlow, tau_copy, lane);
                tau = tau_copy;
                tauE = tau_energy(tau);
            }
            // ---- move on to step t + 1 ----
            Eh = EhNext;
            if ((t & 15u) == 15u) {
                tau = ld_relaxed_u64(&ctrl->tau);
                tauE = tau_energy(tau);
            }
        }
    }
    // ---- unit complete ----
    asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory");
    __syncthreads();
    if (lane == 0 && flagged) {
        atomicAdd(&ctrl->z_flagged, flagged);
        atomicAdd(&ctrl->hits, flagged << (ZB - LOWBITS));               // sixteen blocks of 1024 per flagged block ...
        atomicAdd(&ctrl->false_hits, (flagged << (ZB - LOWBITS)) - sub_true);    // ... of which these held no candidate
    }
    if (tid == 0) {
        atomicAdd(&ctrl->z_steps, (unsigned long long)Z_THREADS << (dead ? 0 : Lw));
        __threadfence();
        if (!dead) atomicAdd(&ctrl->done_configs, 1ull << unit_bits);
    }
    __syncwarp();
    if (warp == 0) {
        asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
        asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, %1;" :: "r"(tmem), "r"(128));
    }
}

// ---- self-test of the one hardware property the screen's proof leans on: a tcgen05 bf16 GEMM of POSITIVE terms with
// fp32 accumulation loses at most a tiny relative amount. One CTA: pseudo-random positive operands spanning many
// binades (A in 2^[-100, 0], T in 2^[-40, 40], like the kernel's), D from the tensor core against the same sums
// formed in fp64 on the CUDA cores from the same bf16 values. out[0] = max over entries of (ref - D) / ref
// (under-estimate), out[1] = max of (D - ref) / ref. ----
__device__ __forceinline__ unsigned zmix(unsigned x) { x ^= x >> 16; x *= 0x7feb352du; x ^= x >> 15; x *= 0x846ca68bu; x ^= x >> 16; return x; }

__global__ void __launch_bounds__(Z_THREADS) zselftest_kernel(unsigned seed, double* __restrict__ out)
{
    extern __shared__ __align__(1024) unsigned char zsmem[];
    unsigned char* sT = zsmem;
    unsigned char* sA = zsmem + 32768;
    __shared__ __align__(8) unsigned long long mbar;
    __shared__ unsigned s_tmem;
    __shared__ double s_under, s_over;
    const int tid = threadIdx.x, warp = tid >> 5;
    if (tid == 0) { s_under = 0.0; s_over = 0.0; }
    // row tid of A (thread's own) and row tid of T (n = tid), K = 128 entries each
    for (int k = 0; k < 128; ++k) {
        const unsigned ha = zmix(seed ^ (unsigned)(tid * 131 + k) * 2654435761u), ht = zmix(ha + 0x9e3779b9u);
        const float va = exp2f(-(float)(ha % 100u) - (float)((ha >> 8) & 1023u) / 1024.f);
        const float vt = exp2f((float)(ht % 81u) - 40.f - (float)((ht >> 8) & 1023u) / 1024.f);
        const unsigned off = (unsigned)(tid >> 3) * Z_SBO + (unsigned)(k >> 3) * Z_LBO + (unsigned)(tid & 7) * 16u + (unsigned)(k & 7) * 2u;
        *reinterpret_cast<__nv_bfloat16*>(sA + off) = __float2bfloat16_rn(va);
        *reinterpret_cast<__nv_bfloat16*>(sT + off) = __float2bfloat16_rn(vt);
    }
    if (tid == 0) {
        asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" :: "r"(smem_u32(&mbar)), "r"(1));
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    if (warp == 0) {
        asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], %1;" :: "r"(smem_u32(&s_tmem)), "r"(128));
        asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;");
    }
    asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
    asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory");
    __syncthreads();
    asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
    const unsigned tmem = s_tmem;
    if (tid == 0) {
        const unsigned a0 = smem_u32(sA), b0 = smem_u32(sT);
#pragma unroll
        for (int ks = 0; ks < 8; ++ks) {
            const unsigned long long da = umma_desc(a0 + (unsigned)ks * 2u * Z_LBO);
            const unsigned long long db = umma_desc(b0 + (unsigned)ks * 2u * Z_LBO);
            const unsigned acc = ks > 0 ? 1u : 0u;
            asm volatile("{\n\t.reg .pred p;\n\tsetp.ne.b32 p, %4, 0;\n\t"
                         "tcgen05.mma.cta_group::1.kind::f16 [%0], %1, %2, %3, p;\n\t}"
                         :: "r"(tmem), "l"(da), "l"(db), "r"(Z_IDESC), "r"(acc) : "memory");
        }
        asm volatile("tcgen05.commit.cta_group::1.mbarrier::arrive::one.shared::cluster.b64 [%0];" :: "r"(smem_u32(&mbar)) : "memory");
    }
    asm volatile("{\n\t.reg .pred P1;\n\tSWAIT_%=:\n\t"
                 "mbarrier.try_wait.parity.shared::cta.b64 P1, [%0], %1;\n\t"
                 "@P1 bra SDONE_%=;\n\tbra SWAIT_%=;\n\tSDONE_%=:\n\t}" :: "r"(smem_u32(&mbar)), "r"(0) : "memory");
    __syncwarp();
    asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
    double under = 0.0, over = 0.0;
    for (int c = 0; c < 4; ++c) {
        unsigned v[32];
        const unsigned taddr = tmem + ((unsigned)(warp * 32) << 16) + (unsigned)(c * 32);
        asm volatile("tcgen05.ld.sync.aligned.32x32b.x32.b32 "
                     "{%0, %1, %2, %3, %4, %5, %6, %7, %8, %9, %10, %11, %12, %13, %14, %15, "
                     "%16, %17, %18, %19, %20, %21, %22, %23, %24, %25, %26, %27, %28, %29, %30, %31}, [%32];"
                     : "=r"(v[0]), "=r"(v[1]), "=r"(v[2]), "=r"(v[3]), "=r"(v[4]), "=r"(v[5]), "=r"(v[6]), "=r"(v[7]),
                       "=r"(v[8]), "=r"(v[9]), "=r"(v[10]), "=r"(v[11]), "=r"(v[12]), "=r"(v[13]), "=r"(v[14]), "=r"(v[15]),
                       "=r"(v[16]), "=r"(v[17]), "=r"(v[18]), "=r"(v[19]), "=r"(v[20]), "=r"(v[21]), "=r"(v[22]), "=r"(v[23]),
                       "=r"(v[24]), "=r"(v[25]), "=r"(v[26]), "=r"(v[27]), "=r"(v[28]), "=r"(v[29]), "=r"(v[30]), "=r"(v[31])
                     : "r"(taddr) : "memory");
        asm volatile("tcgen05.wait::ld.sync.aligned;" ::: "memory");
        for (int j = 0; j < 32; ++j) {
            const int n = c * 32 + j;
            double ref = 0.0;
            for (int k = 0; k < 128; ++k) {
                const unsigned oa = (unsigned)(tid >> 3) * Z_SBO + (unsigned)(k >> 3) * Z_LBO + (unsigned)(tid & 7) * 16u + (unsigned)(k & 7) * 2u;
                const unsigned ot = (unsigned)(n >> 3) * Z_SBO + (unsigned)(k >> 3) * Z_LBO + (unsigned)(n & 7) * 16u + (unsigned)(k & 7) * 2u;
                ref += (double)__bfloat162float(*reinterpret_cast<const __nv_bfloat16*>(sA + oa)) *
                       (double)__bfloat162float(*reinterpret_cast<const __nv_bfloat16*>(sT + ot));
            }
            const double d = (double)__uint_as_float(v[j]);
            if (ref > 0.0) {
                under = fmax(under, (ref - d) / ref);
                over = fmax(over, (d - ref) / ref);
            }
        }
    }
    // positive doubles order like their bit patterns
    atomicMax(reinterpret_cast<unsigned long long*>(&s_under), (unsigned long long)__double_as_longlong(under));
    atomicMax(reinterpret_cast<unsigned long long*>(&s_over), (unsigned long long)__double_as_longlong(over));
    asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory");
    __syncthreads();
    if (tid == 0) { out[0] = s_under; out[1] = s_over; }
    __syncwarp();
    if (warp == 0) {
        asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
        asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, %1;" :: "r"(tmem), "r"(128));
    }
}

void launch_zselftest(unsigned seed, double* out_dev, cudaStream_t st)
{
    cudaFuncSetAttribute(zselftest_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, Z_SMEM_BYTES);
    zselftest_kernel<<<1, Z_THREADS, Z_SMEM_BYTES, st>>>(seed, out_dev);
}

void launch_ztables(const Tables* tab, const Ctrl* ctrl, ZTables* zt, int N, cudaStream_t st)
{
    ztables_kernel<<<1, 1024, 0, st>>>(tab, ctrl, zt, N);
}

void launch_zwalk(const Tables* tab, const ZTables* zt, Ctrl* ctrl, Entry* pool, unsigned* hist, const Plan& plan,
                  cudaStream_t st)
{
    zwalk_kernel<<<(unsigned)plan.total_units, Z_THREADS, Z_SMEM_BYTES, st>>>(tab, zt, ctrl, pool, hist, plan);
}

void set_zscreen_attributes()
{
    cudaFuncSetAttribute(zwalk_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, Z_SMEM_BYTES);
}

}  // namespace ising
