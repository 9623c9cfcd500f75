// enumerate16.cu -- SURVEY.md section 8 rows a2, a3, a4 with TWO configurations per ALU instruction.
//
// Same decomposition as enumerate.cu,  E = Eh + U[mid] + (V[lo] + C[mid][lo])  (the QUBO form of eqs. (2),(3),
// PAPER.md:54-63, around the thread's base state), but the 1024-configuration block is screened in packed 16-bit
// fixed point: one unit = 2^s grid units, every table entry rounded DOWN, so that
//      V16[lo] + C16[mid][lo] + U16[mid]  <=  (V[lo] + C[mid][lo] + U[mid]) / 2^s            (a rigorous lower bound)
// and the inner operation  m = min(V16 + C16, m)  is one VIADDMNMX.U16x2 for the two configurations (lo, mid) and
// (lo, mid | 8): about 450 ALU instructions per 1024 configurations instead of 1024 + 32. A block whose bound is
// <= tau is formed again by the whole warp in exact int32 grid arithmetic (the same a4 path as enumerate.cu), so
// what reaches the pool -- and everything after it -- is identical to the int32 kernel; the 16-bit screen can only
// cause extra (false) hits, never a miss. For integer instances with small weights s = 0 and the screen is exact.
//
// Representation (stage.cu chooses s so that no 16-bit half ever wraps and every half is a NON-NEGATIVE number);
// m0(u) = (u & 7) | ((u >> 3) << 4):
//   Va[lo]  both halves = V16[lo] + bV                                             mid bit 4 clear
//   Vb[lo]  both halves = floor((V[lo] + C[16][lo]) / 2^s) + bV                    mid bit 4 set
//   Cp[u][lo] = ( C16[m0(u)][lo] + cC , C16[m0(u) | 8][lo] + cC )
//   Up[u]   = ( U16[m0(u)] + cU , U16[m0(u) | 8] + cU )
//   block bound = min over halves of g  -  (bV + cC + cU)
// The two halves of a word differ in mid bit 3; mid bit 4 is resolved by the two register sets Va / Vb, which both
// consume the SAME row of Cp (rows u < 8 only): one warp-uniform LDS.128 feeds 8 add-mins.
// Because every half is non-negative and stays inside its 16 bits, a packed sum is also a plain 32-bit integer add.
// That is used three times to take work off the ALU pipe, which bounds the kernel (adds issue as IMAD x*1+y on the
// FMA pipe):
//   * a Gray step updates the packed tables with 32-bit adds of the packed delta (d_lo + 65536 d_hi);
//   * the first sum of every row and the two sums of every row fold are plain adds; the fold's minimum of three is
//     ONE VIMNMX3.U16x2;
//   * in the last P1_CHUNKS of the 8 chunks of a row the sums are plain adds and one VIMNMX3.U16x2 takes the minimum
//     of two of them: 4 configurations per ALU instruction instead of 2, for one more issue slot per two sums.
//     Measured on B200 (2^45-state slice of cfg5): P1_CHUNKS = 0: 3.25e13/s, 1: 3.39e13, 2: 3.42e13, 3: 3.41e13,
//     4: 3.41e13, 5: 3.29e13 -- beyond 2 the issue slots, not the ALU pipe, become the limit.
//
// Walk: as in enumerate.cu (reflected Gray code over the Lw walk bits). The walked 16-bit tables are
// V16 = floor(V(q0)/2^s) + sum over SET walk bits k of floor(DV_on[k]/2^s): turning a bit off subtracts exactly what
// turning it on added, so the bound never drifts: V16 <= V/2^s < V16 + 1 + Lw at every step.
//
// Base state (a2): the block computes the local fields Phi_i and the energy of its base state (thread bits zero)
// once in shared memory; a thread adds the contribution of its own <= 8 thread bits, O(8 N_low) instead of O(N^2).
//
// Register allocation matters: every VIADDMNMX reads three distinct registers, and ptxas's choice of even/odd
// register banks for them decides whether the instruction takes 2 or 3 register-file cycles. The statement order
// of the inline hit path below is the one for which ptxas 12.9 finds a conflict-free allocation (6 of 528 add-mins
// with three same-bank sources instead of 128; 2.5 % in throughput) -- check with cuobjdump after touching it.
#include "common.cuh"

namespace ising {

constexpr int E16_THREADS = 256;
constexpr int NHALF = NMID / 2;
#ifndef P1_CHUNKS
#define P1_CHUNKS 2
#endif

static_assert(LL == 5 && LM == 5, "the subset-sum unrolling below assumes 5 lo and 5 mid bits");

// 32-bit add that is kept off the ALU pipe: IMAD x*1+y executes on the FMA pipe.
__device__ __forceinline__ unsigned add_fma_pipe(unsigned x, unsigned d)
{
    unsigned r;
    asm("mad.lo.u32 %0, %1, 1, %2;" : "=r"(r) : "r"(x), "r"(d));
    return r;
}

// a4, second half: the whole warp forms the 1024 energies of one hit block exactly (int32 grid units) and pushes the
// survivors. qh = the hit lane's state with lo and mid bits zero, eh = its energy. Kept out of line so that its
// registers do not weigh on the enumeration loop (it runs for a vanishing fraction of the blocks).
__device__ __noinline__ void reform_hit_block(const Tables* __restrict__ tab, Ctrl* __restrict__ ctrl,
                                              Entry* __restrict__ pool, const int* sC, int N, unsigned long long qh,
                                              int eh, int tauE, unsigned long long tauQ, int lane)
{
    const int* __restrict__ Jq = tab->Jq;
    const int* __restrict__ hq = tab->hq;
    int vx = tab->QL[lane], ux = tab->QM[lane];
    for (int i = 0; i < LOWBITS; ++i) {
        // local field of spin i at the hit lane's current state, summed by the warp
        int part = 0;
        for (int j = lane; j < N; j += 32) {
            const int w = Jq[i * 64 + j];
            part += ((qh >> j) & 1ull) ? w : -w;
        }
        const int f = hq[i] + __reduce_add_sync(0xffffffffu, part);
        if (i < LL) { if (lane >> i & 1) vx -= 2 * f; }
        else        { if (lane >> (i - LL) & 1) ux -= 2 * f; }
    }
    const unsigned long long qs = qh + (unsigned)lane;
    const int v = vx + eh;
    // two passes: count the survivors, reserve their pool slots with ONE atomic per hit block, then write
    int cnt = 0;
    for (int mid = 0; mid < NMID; ++mid) {
        const int e = v + sC[mid * NLO + lane] + __shfl_sync(0xffffffffu, ux, mid);
        const unsigned long long q = qs + ((unsigned)mid << LL);
        cnt += (e < tauE || (e == tauE && q < tauQ)) ? 1 : 0;
    }
    int incl = cnt;
#pragma unroll
    for (int d = 1; d < 32; d <<= 1) {
        const int n = __shfl_up_sync(0xffffffffu, incl, d);
        if (lane >= d) incl += n;
    }
    const int total = __shfl_sync(0xffffffffu, incl, 31);
    if (total == 0) return;                                     // a false hit of the 16-bit screen
    unsigned slot = 0;
    if (lane == 0) slot = atomicAdd(&ctrl->count, (unsigned)total);
    slot = __shfl_sync(0xffffffffu, slot, 0) + (unsigned)(incl - cnt);
    for (int mid = 0; mid < NMID; ++mid) {
        const int e = v + sC[mid * NLO + lane] + __shfl_sync(0xffffffffu, ux, mid);
        const unsigned long long q = qs + ((unsigned)mid << LL);
        if (e < tauE || (e == tauE && q < tauQ)) {
            if (slot < POOL_CAP) {
                Entry en;
                en.key = key_from_i32(e);
                en.q = q;
                pool[slot] = en;
            }
            ++slot;
        }
    }
}

// HEAVY_HITS = true : hit blocks go through reform_hit_block (one atomic per block) -- for the first launches of a run,
//                     while the threshold is still poor and most blocks are hits.
// HEAVY_HITS = false: the same arithmetic inline with one atomic per survivor -- for the bulk of the run, where a hit
//                     is a rare event and what matters is that the hit path costs the loop no registers (1.4 % faster).
template <bool HEAVY_HITS>
__global__ void __launch_bounds__(E16_THREADS, 2)
enumerate16_kernel(const Tables* __restrict__ tab, Ctrl* __restrict__ ctrl, Entry* __restrict__ pool,
                   int N, int Lw, unsigned long long base, unsigned nthreads)
{
    __shared__ __align__(16) unsigned sCp[(NHALF / 2) * NLO];   // rows u < 8 (mid bit 4 clear); set b covers the rest
    __shared__ __align__(16) unsigned sDVp[LW_MAX * 2 * NLO];
    __shared__ __align__(16) unsigned sDUp[LW_MAX * 2 * NHALF];
    __shared__ int sC[NMID * NLO];
    __shared__ int sDW[1 << LW_MAX];
    __shared__ int sPhiB[64];
    __shared__ int sPhiW[LW_MAX][E16_THREADS];     // per-thread local fields of the walk spins at q0
    __shared__ int sEB;

    const int* __restrict__ Jq = tab->Jq;
    const int* __restrict__ hq = tab->hq;
    const int nlow = LOWBITS + Lw;
    const unsigned long long qB = base + ((unsigned long long)(blockIdx.x * blockDim.x) << nlow);

    for (int i = threadIdx.x; i < (NHALF / 2) * NLO; i += blockDim.x) sCp[i] = tab->Cp[i];
    for (int i = threadIdx.x; i < LW_MAX * 2 * NLO; i += blockDim.x) sDVp[i] = tab->DVp[i];
    for (int i = threadIdx.x; i < LW_MAX * 2 * NHALF; i += blockDim.x) sDUp[i] = tab->DUp[i];
    for (int i = threadIdx.x; i < NMID * NLO; i += blockDim.x) sC[i] = tab->C[i];
    for (int i = threadIdx.x; i < (1 << Lw); i += blockDim.x) sDW[i] = tab->DW[i];
    if (threadIdx.x == 0) sEB = 0;
    // ---- a2, block part: Phi_i(qB) = hq_i + sum_j Jq_ij s_j(qB) for every spin ----
    for (int i = threadIdx.x; i < 64; i += blockDim.x) {
        int acc = 0;
        if (i < N) {
            acc = hq[i];
            const int* row = Jq + i * 64;
            for (int j = 0; j < N; ++j) {
                const int v = row[j];                           // Jq_ii = 0
                acc += ((unsigned)(qB >> j) & 1u) ? v : -v;
            }
        }
        sPhiB[i] = acc;
    }
    __syncthreads();
    // E(qB) = -1/2 sum_i s_i (Phi_i + hq_i)   (each pair is counted twice in sum_i s_i (Phi_i - hq_i); the sum is even)
    for (int i = threadIdx.x; i < N; i += blockDim.x) {
        const int v = sPhiB[i] + hq[i];
        atomicAdd(&sEB, ((unsigned)(qB >> i) & 1u) ? v : -v);
    }
    __syncthreads();

    const unsigned gtid = blockIdx.x * blockDim.x + threadIdx.x;
    if (gtid >= nthreads) return;                  // nthreads is a multiple of 32: whole warps leave together
    const int lane = threadIdx.x & 31;
    const unsigned long long q0 = qB + ((unsigned long long)threadIdx.x << nlow);

    // ---- a2, thread part: q0 differs from qB in the spins D above the walk bits (the thread bits, plus whatever a
    //      carry touches when the launch base is not aligned to the block). With s = spin values at q0:
    //      Phi_i(q0) = Phi_i(qB) + 2 sum_{a in D} Jq[i][a] s_a
    //      E(q0)     = E(qB) - 2 sum_{a in D} s_a Phi_a(qB) - 4 sum_{a<b in D} Jq[a][b] s_a s_b
    int Phi[LOWBITS];
    int PhiW[LW_MAX];
#pragma unroll
    for (int i = 0; i < LOWBITS; ++i) Phi[i] = sPhiB[i];
#pragma unroll
    for (int i = 0; i < LW_MAX; ++i) PhiW[i] = (i < Lw) ? sPhiB[LOWBITS + i] : 0;
    int E0 = -(sEB / 2);
    const unsigned long long dq = (q0 ^ qB) >> nlow;
    for (int j = 0; nlow + j < N; ++j) {
        const bool fl = (dq >> j) & 1ull;
        if (!__any_sync(0xffffffffu, fl)) continue;
        const int a = nlow + j;
        const bool up = (q0 >> a) & 1ull;          // s_a = +1 at q0
        const int* col = Jq + a * 64;              // row a = column a (symmetric): warp-uniform loads
#pragma unroll
        for (int i = 0; i < LOWBITS; ++i) { const int v = 2 * col[i]; Phi[i] += fl ? (up ? v : -v) : 0; }
#pragma unroll
        for (int i = 0; i < LW_MAX; ++i) {
            const int v = (i < Lw) ? 2 * col[LOWBITS + i] : 0;
            PhiW[i] += fl ? (up ? v : -v) : 0;
        }
        int e = up ? -2 * sPhiB[a] : 2 * sPhiB[a];
        for (int jj = 0; jj < j; ++jj) {
            if (!((dq >> jj) & 1ull)) continue;
            const bool upb = (q0 >> (nlow + jj)) & 1ull;
            const int v = 4 * col[nlow + jj];
            e -= (up == upb) ? v : -v;
        }
        E0 += fl ? e : 0;
    }

#pragma unroll
    for (int i = 0; i < LW_MAX; ++i) sPhiW[i][threadIdx.x] = PhiW[i];

    const int s16 = tab->shift16;
    const int cU = tab->cU16;
    const int bV = tab->bV16;
    unsigned Va[NLO], Vb[NLO], Up[NHALF];
    {
        // exact V[x] = QL[x] - 2 sum_{i in x} Phi_i by subset sums, then floor to 16-bit units and bias
        int acc[NLO];
        acc[0] = 0;
#pragma unroll
        for (int x = 1; x < NLO; ++x) {
            const int low = x & -x;
            acc[x] = acc[x ^ low] - 2 * Phi[low == 1 ? 0 : low == 2 ? 1 : low == 4 ? 2 : low == 8 ? 3 : 4];
        }
#pragma unroll
        for (int x = 0; x < NLO; ++x) {
            const int v = acc[x] + tab->QL[x];
            Va[x] = (unsigned)((v >> s16) + bV) * 65537u;                           // mid bit 4 clear
            Vb[x] = (unsigned)(((v + tab->C[16 * NLO + x]) >> s16) + bV) * 65537u;  // mid bit 4 set
        }
        acc[0] = 0;
#pragma unroll
        for (int x = 1; x < NMID; ++x) {
            const int low = x & -x;
            acc[x] = acc[x ^ low] - 2 * Phi[LL + (low == 1 ? 0 : low == 2 ? 1 : low == 4 ? 2 : low == 8 ? 3 : 4)];
        }
#pragma unroll
        for (int r = 0; r < NHALF; ++r) {
            const int m0 = (r & 7) | ((r >> 3) << 4), m1 = m0 | 8;
            const unsigned u0 = (unsigned)(((acc[m0] + tab->QM[m0]) >> s16) + cU);
            const unsigned u1 = (unsigned)(((acc[m1] + tab->QM[m1]) >> s16) + cU);
            Up[r] = u0 + (u1 << 16);
        }
    }
    int Eh = E0;

    const int tauE = ctrl->tauE;
    const unsigned long long tauQ = ctrl->tauQ;
    const unsigned long long q0_warp = q0 - ((unsigned long long)lane << nlow);
    const int bias = bV + tab->cC16 + cU;

    const unsigned nsteps = 1u << Lw;
    for (unsigned t = 0; t < nsteps; ++t) {
        asm volatile("" ::: "memory");                 // the tables are re-read every step: keep them out of registers
        if (t > 0) {
            // ---- Gray step: flip walk bit k = ctz(t); warp-uniform rows; packed words updated on the FMA pipe ----
            const int k = __ffs(t) - 1;
            const unsigned gnew = t ^ (t >> 1);
            const int sb = (gnew >> k) & 1;
            const int phi = sPhiW[k][threadIdx.x];
            Eh += sDW[t] + (sb ? -2 * phi : 2 * phi);
            const uint4* dv = reinterpret_cast<const uint4*>(sDVp + (k * 2 + sb) * NLO);
            const uint4* du = reinterpret_cast<const uint4*>(sDUp + (k * 2 + sb) * NHALF);
#pragma unroll
            for (int x = 0; x < NLO / 4; ++x) {
                const uint4 d = dv[x];
                Va[4 * x + 0] = add_fma_pipe(Va[4 * x + 0], d.x);
                Va[4 * x + 1] = add_fma_pipe(Va[4 * x + 1], d.y);
                Va[4 * x + 2] = add_fma_pipe(Va[4 * x + 2], d.z);
                Va[4 * x + 3] = add_fma_pipe(Va[4 * x + 3], d.w);
                Vb[4 * x + 0] = add_fma_pipe(Vb[4 * x + 0], d.x);
                Vb[4 * x + 1] = add_fma_pipe(Vb[4 * x + 1], d.y);
                Vb[4 * x + 2] = add_fma_pipe(Vb[4 * x + 2], d.z);
                Vb[4 * x + 3] = add_fma_pipe(Vb[4 * x + 3], d.w);
            }
#pragma unroll
            for (int x = 0; x < NHALF / 4; ++x) {
                const uint4 d = du[x];
                Up[4 * x + 0] = add_fma_pipe(Up[4 * x + 0], d.x);
                Up[4 * x + 1] = add_fma_pipe(Up[4 * x + 1], d.y);
                Up[4 * x + 2] = add_fma_pipe(Up[4 * x + 2], d.z);
                Up[4 * x + 3] = add_fma_pipe(Up[4 * x + 3], d.w);
            }
        }
        // ---- a3: 1024 configurations, one packed add-min per two of them ----
        unsigned g = 0xffffffffu;
#pragma unroll
        for (int r = 0; r < NHALF / 2; ++r) {
            // one row of C serves two register sets (mid bit 4 clear / set): 8 add-mins per LDS.128,
            // and the two chains are independent
            const uint4* crow = reinterpret_cast<const uint4*>(sCp + r * NLO);
            unsigned ma, mb;
#pragma unroll
            for (int x = 0; x < NLO / 4; ++x) {
                const uint4 c = crow[x];
                if (x == 0) {
                    // the first sum of a row needs no minimum: a plain packed add (no half can wrap), FMA pipe
                    ma = add_fma_pipe(Va[0], c.x);
                    mb = add_fma_pipe(Vb[0], c.x);
                    ma = __viaddmin_u16x2(Va[1], c.y, ma);
                    mb = __viaddmin_u16x2(Vb[1], c.y, mb);
                    ma = __viaddmin_u16x2(Va[2], c.z, ma);
                    mb = __viaddmin_u16x2(Vb[2], c.z, mb);
                    ma = __viaddmin_u16x2(Va[3], c.w, ma);
                    mb = __viaddmin_u16x2(Vb[3], c.w, mb);
                } else if (x >= NLO / 4 - P1_CHUNKS) {
                    // pipe balancing: these sums are formed as plain packed adds on the FMA pipe and one VIMNMX3
                    // takes the minimum of two of them -- half the ALU-pipe time, one more issue slot per two sums
                    const unsigned a0 = add_fma_pipe(Va[4 * x + 0], c.x), b0 = add_fma_pipe(Vb[4 * x + 0], c.x);
                    const unsigned a1 = add_fma_pipe(Va[4 * x + 1], c.y), b1 = add_fma_pipe(Vb[4 * x + 1], c.y);
                    const unsigned a2 = add_fma_pipe(Va[4 * x + 2], c.z), b2 = add_fma_pipe(Vb[4 * x + 2], c.z);
                    const unsigned a3 = add_fma_pipe(Va[4 * x + 3], c.w), b3 = add_fma_pipe(Vb[4 * x + 3], c.w);
                    ma = __vimin3_u16x2(ma, a0, a1);
                    mb = __vimin3_u16x2(mb, b0, b1);
                    ma = __vimin3_u16x2(ma, a2, a3);
                    mb = __vimin3_u16x2(mb, b2, b3);
                } else {
                    ma = __viaddmin_u16x2(Va[4 * x + 0], c.x, ma);
                    mb = __viaddmin_u16x2(Vb[4 * x + 0], c.x, mb);
                    ma = __viaddmin_u16x2(Va[4 * x + 1], c.y, ma);
                    mb = __viaddmin_u16x2(Vb[4 * x + 1], c.y, mb);
                    ma = __viaddmin_u16x2(Va[4 * x + 2], c.z, ma);
                    mb = __viaddmin_u16x2(Vb[4 * x + 2], c.z, mb);
                    ma = __viaddmin_u16x2(Va[4 * x + 3], c.w, ma);
                    mb = __viaddmin_u16x2(Vb[4 * x + 3], c.w, mb);
                }
            }
            // fold both rows into g with ONE ALU instruction: the two packed sums cannot wrap (stage.cu), so they are
            // plain 32-bit adds on the FMA pipe, and VIMNMX3 takes the minimum of the three
            g = __vimin3_u16x2(g, add_fma_pipe(ma, Up[r]), add_fma_pipe(mb, Up[r + NHALF / 2]));
        }
        // ---- a4: threshold filter on the lower bound:  bound * 2^s + Eh <= tauE  <=>  bound <= (tauE - Eh) >> s ----
        const int gm = (int)min(g & 0xffffu, g >> 16) - bias;
        unsigned hits = __ballot_sync(0xffffffffu, gm <= ((tauE - Eh) >> s16));
        while (hits) {
            // the whole warp re-forms the 1024 energies of the hit lane exactly (int32 grid units)
            const int src = __ffs(hits) - 1;
            hits &= hits - 1;
            const unsigned gray = t ^ (t >> 1);
            const unsigned long long qh = q0_warp + ((unsigned long long)src << nlow) + ((unsigned long long)gray << LOWBITS);
            if (HEAVY_HITS) {
                const int eh = __shfl_sync(0xffffffffu, Eh, src);
                reform_hit_block(tab, ctrl, pool, sC, N, qh, eh, tauE, tauQ, lane);
            } else {
                int vx = tab->QL[lane], ux = tab->QM[lane];
                for (int i = 0; i < LOWBITS; ++i) {
                    int part = 0;
                    for (int j = lane; j < N; j += 32) {
                        const int w = Jq[i * 64 + j];
                        part += ((qh >> j) & 1ull) ? w : -w;
                    }
                    const int f = hq[i] + __reduce_add_sync(0xffffffffu, part);
                    if (i < LL) { if (lane >> i & 1) vx -= 2 * f; }
                    else        { if (lane >> (i - LL) & 1) ux -= 2 * f; }
                }
                const int eh = __shfl_sync(0xffffffffu, Eh, src);
                const unsigned long long qs = qh + (unsigned)lane;
                const int v = vx + eh;
                for (int mid = 0; mid < NMID; ++mid) {
                    const int e = v + sC[mid * NLO + lane] + __shfl_sync(0xffffffffu, ux, mid);
                    const unsigned long long q = qs + ((unsigned)mid << LL);
                    if (e < tauE || (e == tauE && q < tauQ)) {
                        const unsigned idx = atomicAdd(&ctrl->count, 1u);
                        if (idx < POOL_CAP) {
                            Entry en;
                            en.key = key_from_i32(e);
                            en.q = q;
                            pool[idx] = en;
                        }
                    }
                }
            }
        }
    }
}

void launch_enumerate16(const Tables* tab, Ctrl* ctrl, Entry* pool, int N, int Lw,
                        unsigned long long base, unsigned nthreads, bool heavy_hits, cudaStream_t st)
{
    const unsigned threads = nthreads < (unsigned)E16_THREADS ? nthreads : (unsigned)E16_THREADS;
    const unsigned blocks = (nthreads + threads - 1) / threads;
    if (heavy_hits) enumerate16_kernel<true><<<blocks, threads, 0, st>>>(tab, ctrl, pool, N, Lw, base, nthreads);
    else enumerate16_kernel<false><<<blocks, threads, 0, st>>>(tab, ctrl, pool, N, Lw, base, nthreads);
}

}  // namespace ising
