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
//   * in three of the 8 chunks of a row (E16_P1MASK) the sums are plain adds and one VIMNMX3.U16x2 takes the minimum
//     of two of them: 4 configurations per ALU instruction instead of 2, for one more issue slot per two sums.
//     The measured rate of this instruction mix in isolation (ising_addmin_mix_peak) is NOT above the fused form's
//     (VIMNMX3.U16x2 issues at the same 2 cycles per warp as VIADDMNMX.U16x2 and does not overlap with it); what
//     the split chunks buy is scheduling slack, a few per cent (table in hit_step below).
//
// Walk: as in enumerate.cu (reflected Gray code over the Lw walk bits). The walked 16-bit tables are
// V16 = floor(V(q0)/2^s) + sum over SET walk bits k of floor(DV_on[k]/2^s): turning a bit off subtracts exactly what
// turning it on added, so the bound never drifts: V16 <= V/2^s < V16 + 1 + Lw at every step.
//
// Base state (a2), work distribution and the exact forming of hit blocks are in walk.cuh (the persistent kernel this
// file instantiates): a warp computes the local fields and the energy of its unit's first state once, a lane adds the
// contribution of its own 5 lane bits.
//
// Register allocation matters: every VIADDMNMX reads three distinct registers, and ptxas's choice of even/odd
// register banks for them decides whether the instruction takes 2 or 3 register-file cycles. The statement order
// of the inline hit path below is the one for which ptxas 12.9 finds a conflict-free allocation (6 of 528 add-mins
// with three same-bank sources instead of 128; 2.5 % in throughput) -- check with cuobjdump after touching it.
#include "walk.cuh"

namespace ising {

constexpr int NHALF = NMID / 2;

static_assert(LL == 5 && LM == 5, "the subset-sum unrolling below assumes 5 lo and 5 mid bits");

// 32-bit add that is kept off the ALU pipe: IMAD x*1+y executes on the FMA pipe.
__device__ __forceinline__ unsigned add_fma_pipe(unsigned x, unsigned d)
{
    unsigned r;
    asm("mad.lo.u32 %0, %1, 1, %2;" : "=r"(r) : "r"(x), "r"(d));
    return r;
}

struct Inner16 {
    struct Shared {
        __align__(16) unsigned Cp[(NHALF / 2) * NLO];   // rows u < 8 (mid bit 4 clear); register set b covers the rest
        __align__(16) unsigned DVp[LW_MAX * 2 * NLO];
        __align__(16) unsigned DUp[LW_MAX * 2 * NHALF];
    };
    struct Regs {
        unsigned Va[NLO], Vb[NLO], Up[NHALF];
        int bias, s16;
    };

    static __device__ __forceinline__ void load_shared(Shared& sh, const Tables* __restrict__ tab)
    {
        for (int i = threadIdx.x; i < (NHALF / 2) * NLO; i += blockDim.x) sh.Cp[i] = tab->Cp[i];
        for (int i = threadIdx.x; i < LW_MAX * 2 * NLO; i += blockDim.x) sh.DVp[i] = tab->DVp[i];
        for (int i = threadIdx.x; i < LW_MAX * 2 * NHALF; i += blockDim.x) sh.DUp[i] = tab->DUp[i];
    }

    // exact V[x] = QL[x] - 2 sum_{i in x} Phi_i by subset sums, then floor to 16-bit units and bias
    static __device__ __forceinline__ void init(Regs& R, const Tables* __restrict__ tab, const int (&Phi)[LOWBITS])
    {
        const int s16 = tab->shift16, cU = tab->cU16, bV = tab->bV16;
        R.bias = bV + tab->cC16 + cU;
        R.s16 = s16;
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
            R.Va[x] = (unsigned)((v >> s16) + bV) * 65537u;                           // mid bit 4 clear
            R.Vb[x] = (unsigned)(((v + tab->C[16 * NLO + x]) >> s16) + bV) * 65537u;  // mid bit 4 set
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
            R.Up[r] = u0 + (u1 << 16);
        }
    }

    // a3: 1024 configurations, one packed add-min per two of them; a4: the screen on the lower bound,
    //   bound * 2^s + Eh <= tauE  <=>  bound <= (tauE - Eh) >> s
    // Which of the chunks 1..7 of a row use the split form (bit x of E16_P1MASK), and the statement order of the two
    // register sets inside a fused chunk, decide how ptxas schedules the loop. Measured on B200, 2^43-state slice of
    // cfg5, configurations/s (all variants have 0 register-bank conflicts; order 0 = a then b per word of C, the default
    // of the mask sweep; order 1 = b then a per word, the one kept below; order 2 = all of a, then all of b; two mixed
    // orders, a first where C sits in an even register and the reverse, were no better and are not listed):
    //   mask 0xC0: 3.34e13   0x06: 3.39e13   0x82: 3.36e13   0x60: 3.25e13   0x80: 3.27e13   0xE0: 3.42e13   0x46: 3.40e13
    //   0x1E: 3.37e13   0xF0: 3.29e13   0xAA: 3.30e13   0xE0 + order 1: 3.45e13 (kept)   0xE0 + order 2: 3.41e13
#ifndef E16_P1MASK
#define E16_P1MASK 0xE0          // chunks 5, 6 and 7 of every row in the split form
#endif
    // ... and the Gray step that follows (walk bit k turns on/off): the V tables are updated chunk by chunk right after
    // their last use in the last row, so that the 80 table adds and their loads overlap the add-mins instead of forming
    // a phase of their own at the head of the next step (ncu: a quarter of the stall samples sat at the step boundary).
    static __device__ __forceinline__ bool hit_step(Regs& R, const Shared& sh, const Tables* __restrict__ tab,
                                                    int tauE, int Eh, int k, int sb)
    {
        const uint4* dv = reinterpret_cast<const uint4*>(sh.DVp + (k * 2 + sb) * NLO);
        const uint4* du = reinterpret_cast<const uint4*>(sh.DUp + (k * 2 + sb) * NHALF);
        unsigned g = 0xffffffffu;
#pragma unroll
        for (int r = 0; r < NHALF / 2; ++r) {
            // one row of C serves two register sets (mid bit 4 clear / set): 8 add-mins per LDS.128,
            // and the two chains are independent
            const uint4* crow = reinterpret_cast<const uint4*>(sh.Cp + r * NLO);
            unsigned ma, mb;
#pragma unroll
            for (int x = 0; x < NLO / 4; ++x) {
                const uint4 c = crow[x];
                if (x == 0) {
                    // the first sum of a row needs no minimum: a plain packed add (no half can wrap), FMA pipe
                    ma = add_fma_pipe(R.Va[0], c.x);
                    mb = add_fma_pipe(R.Vb[0], c.x);
                    ma = __viaddmin_u16x2(R.Va[1], c.y, ma);
                    mb = __viaddmin_u16x2(R.Vb[1], c.y, mb);
                    ma = __viaddmin_u16x2(R.Va[2], c.z, ma);
                    mb = __viaddmin_u16x2(R.Vb[2], c.z, mb);
                    ma = __viaddmin_u16x2(R.Va[3], c.w, ma);
                    mb = __viaddmin_u16x2(R.Vb[3], c.w, mb);
                } else if ((E16_P1MASK >> x) & 1) {
                    // pipe balancing: these sums are formed as plain packed adds on the FMA pipe and one VIMNMX3
                    // takes the minimum of two of them
                    const unsigned a0 = add_fma_pipe(R.Va[4 * x + 0], c.x), b0 = add_fma_pipe(R.Vb[4 * x + 0], c.x);
                    const unsigned a1 = add_fma_pipe(R.Va[4 * x + 1], c.y), b1 = add_fma_pipe(R.Vb[4 * x + 1], c.y);
                    const unsigned a2 = add_fma_pipe(R.Va[4 * x + 2], c.z), b2 = add_fma_pipe(R.Vb[4 * x + 2], c.z);
                    const unsigned a3 = add_fma_pipe(R.Va[4 * x + 3], c.w), b3 = add_fma_pipe(R.Vb[4 * x + 3], c.w);
                    ma = __vimin3_u16x2(ma, a0, a1);
                    mb = __vimin3_u16x2(mb, b0, b1);
                    ma = __vimin3_u16x2(ma, a2, a3);
                    mb = __vimin3_u16x2(mb, b2, b3);
                } else {
                    // fused chunk, register set b before set a for every word of C (order 1 of the table above)
                    mb = __viaddmin_u16x2(R.Vb[4 * x + 0], c.x, mb);
                    ma = __viaddmin_u16x2(R.Va[4 * x + 0], c.x, ma);
                    mb = __viaddmin_u16x2(R.Vb[4 * x + 1], c.y, mb);
                    ma = __viaddmin_u16x2(R.Va[4 * x + 1], c.y, ma);
                    mb = __viaddmin_u16x2(R.Vb[4 * x + 2], c.z, mb);
                    ma = __viaddmin_u16x2(R.Va[4 * x + 2], c.z, ma);
                    mb = __viaddmin_u16x2(R.Vb[4 * x + 3], c.w, mb);
                    ma = __viaddmin_u16x2(R.Va[4 * x + 3], c.w, ma);
                }
                if (r == NHALF / 2 - 1) {
                    // last row: this chunk of V is not needed any more in this step
                    const uint4 d = dv[x];
                    R.Va[4 * x + 0] = add_fma_pipe(R.Va[4 * x + 0], d.x);
                    R.Vb[4 * x + 0] = add_fma_pipe(R.Vb[4 * x + 0], d.x);
                    R.Va[4 * x + 1] = add_fma_pipe(R.Va[4 * x + 1], d.y);
                    R.Vb[4 * x + 1] = add_fma_pipe(R.Vb[4 * x + 1], d.y);
                    R.Va[4 * x + 2] = add_fma_pipe(R.Va[4 * x + 2], d.z);
                    R.Vb[4 * x + 2] = add_fma_pipe(R.Vb[4 * x + 2], d.z);
                    R.Va[4 * x + 3] = add_fma_pipe(R.Va[4 * x + 3], d.w);
                    R.Vb[4 * x + 3] = add_fma_pipe(R.Vb[4 * x + 3], d.w);
                }
            }
            // fold both rows into g with ONE ALU instruction: the two packed sums cannot wrap (stage.cu), so they are
            // plain 32-bit adds on the FMA pipe, and VIMNMX3 takes the minimum of the three
            g = __vimin3_u16x2(g, add_fma_pipe(ma, R.Up[r]), add_fma_pipe(mb, R.Up[r + NHALF / 2]));
        }
#pragma unroll
        for (int x = 0; x < NHALF / 4; ++x) {
            const uint4 d = du[x];
            R.Up[4 * x + 0] = add_fma_pipe(R.Up[4 * x + 0], d.x);
            R.Up[4 * x + 1] = add_fma_pipe(R.Up[4 * x + 1], d.y);
            R.Up[4 * x + 2] = add_fma_pipe(R.Up[4 * x + 2], d.z);
            R.Up[4 * x + 3] = add_fma_pipe(R.Up[4 * x + 3], d.w);
        }
        const int gm = (int)min(g & 0xffffu, g >> 16) - R.bias;
        return gm <= ((tauE - Eh) >> R.s16);
    }
};

void launch_walk16(const Tables* tab, Ctrl* ctrl, Entry* pool, unsigned* hist, const Plan& plan, cudaStream_t st)
{
    // one warp per unit of the plan (the queue hands the units out in ascending q whatever the block order)
    const unsigned long long blocks = (plan.total_units + WALK_WARPS - 1) / WALK_WARPS;
    walk_kernel<Inner16><<<(unsigned)blocks, WALK_THREADS, 0, st>>>(tab, ctrl, pool, hist, plan);
}

}  // namespace ising
