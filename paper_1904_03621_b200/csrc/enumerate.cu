// enumerate.cu -- SURVEY.md section 8 rows a2 (base state), a3 (enumeration) and a4 (threshold filter), int32 variant,
// and the direct kernel for tiny instances.
//
// Every configuration's grid energy is formed exactly once, as   E = Eh + U[mid] + (V[lo] + C[mid][lo]),
// the QUBO decomposition of eqs. (2),(3) around the thread's base state q0:
//   V[lo]      per thread, 32 registers : energy change of setting the lo bits (incl. coupling to walk/thread spins)
//   U[mid]     per thread, 32 registers : same for the mid bits
//   C[mid][lo] per instance, shared mem : coupling between lo and mid bits, streamed as warp-uniform LDS.128
//   Eh         per thread scalar        : energy of q0 with the current walk bits
// The inner operation is one VIADDMNMX per configuration:  m = min(V[lo] + C[mid][lo], m)  -- the running
// minimum of a 32-configuration row; rows fold into g = min(m + U[mid], g). Only if g + Eh <= tau (the
// running S-th best, broadcast from global memory) the 1024 energies of that block are formed again by the
// whole warp and the survivors pushed to the candidate pool. With a warm threshold that is a few thousand
// pushes out of 2^N configurations: no per-configuration HBM traffic at all.
//
// Walk (north_star (a), Gray code): the thread's Lw walk bits advance in reflected Gray order; flipping walk bit k
// adds a warp-uniform row DV[k][.] to V, DU[k][.] to U, and DW[t] -+ 2 Phi_k to Eh (the O(N) local-field
// update of the classic Gray walk, restricted to the 64 table entries that depend on bit k).
//
// This is the arithmetic "no narrower than the paper's" (32-bit, exact): the default kernel (enumerate16.cu) screens
// in 16 bits and reaches the same candidate set. Selected with ISING_KERNEL=32; work distribution, base state and
// the exact forming of hit blocks are shared with it (walk.cuh).
#include "walk.cuh"

namespace ising {

struct Inner32 {
    struct Shared {
        __align__(16) int C[NMID * NLO];
        __align__(16) int DV[LW_MAX * 2 * NLO];
        __align__(16) int DU[LW_MAX * 2 * NMID];
    };
    struct Regs {
        int V[NLO], U[NMID];
    };

    static __device__ __forceinline__ void load_shared(Shared& sh, const Tables* __restrict__ tab)
    {
        for (int i = threadIdx.x; i < NMID * NLO; i += blockDim.x) sh.C[i] = tab->C[i];
        for (int i = threadIdx.x; i < LW_MAX * 2 * NLO; i += blockDim.x) sh.DV[i] = tab->DV[i];
        for (int i = threadIdx.x; i < LW_MAX * 2 * NMID; i += blockDim.x) sh.DU[i] = tab->DU[i];
    }

    static __device__ __forceinline__ void init(Regs& R, const Tables* __restrict__ tab, const int (&Phi)[LOWBITS])
    {
#pragma unroll
        for (int x = 0; x < NLO; ++x) {
            int a = tab->QL[x];
#pragma unroll
            for (int i = 0; i < LL; ++i) if (x >> i & 1) a -= 2 * Phi[i];
            R.V[x] = a;
        }
#pragma unroll
        for (int x = 0; x < NMID; ++x) {
            int a = tab->QM[x];
#pragma unroll
            for (int j = 0; j < LM; ++j) if (x >> j & 1) a -= 2 * Phi[LL + j];
            R.U[x] = a;
        }
    }

    static __device__ __forceinline__ void step(Regs& R, const Shared& sh, int k, int sb)
    {
        const int4* dv = reinterpret_cast<const int4*>(sh.DV + (k * 2 + sb) * NLO);
        const int4* du = reinterpret_cast<const int4*>(sh.DU + (k * 2 + sb) * NMID);
#pragma unroll
        for (int x = 0; x < NLO / 4; ++x) {
            const int4 d = dv[x];
            R.V[4 * x + 0] += d.x; R.V[4 * x + 1] += d.y; R.V[4 * x + 2] += d.z; R.V[4 * x + 3] += d.w;
        }
#pragma unroll
        for (int x = 0; x < NMID / 4; ++x) {
            const int4 d = du[x];
            R.U[4 * x + 0] += d.x; R.U[4 * x + 1] += d.y; R.U[4 * x + 2] += d.z; R.U[4 * x + 3] += d.w;
        }
    }

    // a3: 1024 configurations, one add-min each; a4: threshold filter on the exact block minimum; then the Gray step
    static __device__ __forceinline__ bool hit_step(Regs& R, const Shared& sh, const Tables* __restrict__,
                                                    int tauE, int Eh, int k, int sb)
    {
        int g = 0x7fffffff;
#pragma unroll
        for (int mid = 0; mid < NMID; ++mid) {
            const int4* crow = reinterpret_cast<const int4*>(sh.C + mid * NLO);
            int m = 0x7fffffff;
#pragma unroll
            for (int x = 0; x < NLO / 4; ++x) {
                const int4 c = crow[x];
                m = __viaddmin_s32(R.V[4 * x + 0], c.x, m);
                m = __viaddmin_s32(R.V[4 * x + 1], c.y, m);
                m = __viaddmin_s32(R.V[4 * x + 2], c.z, m);
                m = __viaddmin_s32(R.V[4 * x + 3], c.w, m);
            }
            g = __viaddmin_s32(m, R.U[mid], g);
        }
        step(R, sh, k, sb);
        return g <= tauE - Eh;
    }
};

void launch_walk32(const Tables* tab, Ctrl* ctrl, Entry* pool, unsigned* hist, const Plan& plan, cudaStream_t st)
{
    // one warp per unit of the plan (the queue hands the units out in ascending q whatever the block order)
    const unsigned long long blocks = (plan.total_units + WALK_WARPS - 1) / WALK_WARPS;
    walk_kernel<Inner32><<<(unsigned)blocks, WALK_THREADS, 0, st>>>(tab, ctrl, pool, hist, plan);
}

// Direct evaluation of eq. (1) on the grid for every state of a tiny instance (N <= N_DIRECT_MAX, 2^N <= 16384
// states): everything goes to the pool (and, in the single-pass path, to the histogram; the last block to finish
// derives the threshold from it).
__global__ void direct_kernel(const Tables* __restrict__ tab, Ctrl* __restrict__ ctrl, Entry* __restrict__ pool,
                              unsigned* __restrict__ hist, int N, int S, unsigned count, int use_hist)
{
    if (ctrl->status != 0) return;
    const long long Wq = ctrl->Wq;
    const int hs = ctrl->hist_shift;
    for (unsigned t = blockIdx.x * blockDim.x + threadIdx.x; t < count; t += gridDim.x * blockDim.x) {
        const unsigned long long q = t;
        int e = 0;
        for (int i = 0; i < N; ++i) {
            const unsigned bi = (unsigned)(q >> i) & 1u;
            for (int j = i + 1; j < N; ++j) {
                const int v = tab->Jq[i * 64 + j];
                e += (bi ^ ((unsigned)(q >> j) & 1u)) ? v : -v;
            }
            const int hv = tab->hq[i];
            e += bi ? -hv : hv;
        }
        Entry en;
        en.key = key_from_i32(e);
        en.q = q;
        pool[t] = en;
        if (use_hist) {
            const int b = hist_bin(e, Wq, hs);
            atomicAdd(hist + HIST_COARSE + b, 1u);
            atomicAdd(hist + (b >> 8), 1u);
        }
    }
    if (blockIdx.x == 0 && threadIdx.x == 0) ctrl->count = count;
    if (!use_hist) return;
    // the last block to finish turns the histogram into the threshold
    __shared__ int s_last;
    __threadfence();
    __syncthreads();
    if (threadIdx.x == 0) s_last = atomicAdd(&ctrl->blocks_done, 1u) == gridDim.x - 1;
    __syncthreads();
    if (!s_last || threadIdx.x >= 32) return;
    __threadfence();
    int tauE;
    if (hist_threshold(ctrl, hist, (unsigned)S, threadIdx.x, tauE) && threadIdx.x == 0)
        atomicMin(&ctrl->tau, tau_pack(tauE, QC_NONE));
}

void launch_direct(const Tables* tab, Ctrl* ctrl, Entry* pool, unsigned* hist, int N, int S, unsigned count,
                   int use_hist, cudaStream_t st)
{
    const unsigned threads = 128, blocks = (count + threads - 1) / threads;
    direct_kernel<<<blocks, threads, 0, st>>>(tab, ctrl, pool, hist, N, S, count, use_hist);
}

}  // namespace ising
