// enumerate.cu -- SURVEY.md section 8 rows a2 (thread base state), a3 (enumeration) and a4 (threshold filter).
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
#include "common.cuh"

namespace ising {

__device__ __forceinline__ void push_candidate(Ctrl* ctrl, Entry* pool, int e, unsigned long long q)
{
    unsigned idx = atomicAdd(&ctrl->count, 1u);
    if (idx < POOL_CAP) {
        Entry en;
        en.key = key_from_i32(e);
        en.q = q;
        pool[idx] = en;
    }
}

constexpr int ENUM_THREADS = 256;

__global__ void __launch_bounds__(ENUM_THREADS, 2)
enumerate_kernel(const Tables* __restrict__ tab, Ctrl* __restrict__ ctrl, Entry* __restrict__ pool,
                 int N, int Lw, unsigned long long base, unsigned nthreads)
{
    __shared__ __align__(16) int sC[NMID * NLO];
    __shared__ __align__(16) int sDV[LW_MAX * 2 * NLO];
    __shared__ __align__(16) int sDU[LW_MAX * 2 * NMID];
    __shared__ int sDW[1 << LW_MAX];
    __shared__ int sScratch[ENUM_THREADS / 32][NLO + NMID];

    for (int i = threadIdx.x; i < NMID * NLO; i += blockDim.x) sC[i] = tab->C[i];
    for (int i = threadIdx.x; i < LW_MAX * 2 * NLO; i += blockDim.x) sDV[i] = tab->DV[i];
    for (int i = threadIdx.x; i < LW_MAX * 2 * NMID; i += blockDim.x) sDU[i] = tab->DU[i];
    for (int i = threadIdx.x; i < (1 << Lw); i += blockDim.x) sDW[i] = tab->DW[i];
    __syncthreads();

    const unsigned gtid = blockIdx.x * blockDim.x + threadIdx.x;
    if (gtid >= nthreads) return;                  // nthreads is a multiple of 32: whole warps leave together
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const int nlow = LOWBITS + Lw;
    const unsigned long long q0 = base + ((unsigned long long)gtid << nlow);

    // ---- a2: base state. E0 = E(q0) by eq. (1); Phi_i(q0) = hq_i + sum_j Jq_ij s_j(q0) for the L, M, W spins ----
    const int* __restrict__ Jq = tab->Jq;
    const int* __restrict__ hq = tab->hq;
    int E0 = 0;
    for (int i = 0; i < N; ++i) {
        const unsigned bi = (unsigned)(q0 >> i) & 1u;
        const int* row = Jq + i * 64;
        int acc = 0;
        for (int j = i + 1; j < N; ++j) {
            const unsigned bj = (unsigned)(q0 >> j) & 1u;
            const int v = row[j];
            acc += (bi ^ bj) ? v : -v;             // -J s_i s_j
        }
        const int hv = hq[i];
        E0 += acc + (bi ? -hv : hv);               // -h s_i
    }
    int Phi[LOWBITS];
    int PhiW[LW_MAX];
#pragma unroll
    for (int i = 0; i < LOWBITS + LW_MAX; ++i) {
        int acc = 0;
        if (i < nlow && i < N) {
            const int* row = Jq + i * 64;
            acc = hq[i];
            for (int j = 0; j < N; ++j) {
                const int v = row[j];              // Jq_ii = 0
                acc += ((unsigned)(q0 >> j) & 1u) ? v : -v;
            }
        }
        if (i < LOWBITS) Phi[i] = acc; else PhiW[i - LOWBITS] = acc;
    }
    int V[NLO], U[NMID];
#pragma unroll
    for (int x = 0; x < NLO; ++x) {
        int a = tab->QL[x];
#pragma unroll
        for (int i = 0; i < LL; ++i) if (x >> i & 1) a -= 2 * Phi[i];
        V[x] = a;
    }
#pragma unroll
    for (int x = 0; x < NMID; ++x) {
        int a = tab->QM[x];
#pragma unroll
        for (int j = 0; j < LM; ++j) if (x >> j & 1) a -= 2 * Phi[LL + j];
        U[x] = a;
    }
    int Eh = E0;

    const int tauE = ctrl->tauE;
    const unsigned long long tauQ = ctrl->tauQ;
    int* scratch = sScratch[warp];
    const unsigned long long q0_warp = q0 - ((unsigned long long)lane << nlow);

    const unsigned nsteps = 1u << Lw;
    for (unsigned t = 0; t < nsteps; ++t) {
        if (t > 0) {
            // ---- Gray step: flip walk bit k = ctz(t); warp-uniform rows, exact integer updates ----
            const int k = __ffs(t) - 1;
            const unsigned gnew = t ^ (t >> 1);
            const int sb = (gnew >> k) & 1;
            int phi = PhiW[0];
#pragma unroll
            for (int kk = 1; kk < LW_MAX; ++kk) phi = (k == kk) ? PhiW[kk] : phi;
            Eh += sDW[t] + (sb ? -2 * phi : 2 * phi);
            const int4* dv = reinterpret_cast<const int4*>(sDV + (k * 2 + sb) * NLO);
            const int4* du = reinterpret_cast<const int4*>(sDU + (k * 2 + sb) * NMID);
#pragma unroll
            for (int x = 0; x < NLO / 4; ++x) {
                const int4 d = dv[x];
                V[4 * x + 0] += d.x; V[4 * x + 1] += d.y; V[4 * x + 2] += d.z; V[4 * x + 3] += d.w;
            }
#pragma unroll
            for (int x = 0; x < NMID / 4; ++x) {
                const int4 d = du[x];
                U[4 * x + 0] += d.x; U[4 * x + 1] += d.y; U[4 * x + 2] += d.z; U[4 * x + 3] += d.w;
            }
        }
        // ---- a3: 1024 configurations, one add-min each ----
        int g = 0x7fffffff;
#pragma unroll
        for (int mid = 0; mid < NMID; ++mid) {
            const int4* crow = reinterpret_cast<const int4*>(sC + mid * NLO);
            int m = 0x7fffffff;
#pragma unroll
            for (int x = 0; x < NLO / 4; ++x) {
                const int4 c = crow[x];
                m = __viaddmin_s32(V[4 * x + 0], c.x, m);
                m = __viaddmin_s32(V[4 * x + 1], c.y, m);
                m = __viaddmin_s32(V[4 * x + 2], c.z, m);
                m = __viaddmin_s32(V[4 * x + 3], c.w, m);
            }
            g = __viaddmin_s32(m, U[mid], g);
        }
        // ---- a4: threshold filter; survivors are re-formed by the whole warp, one hit lane at a time ----
        unsigned hits = __ballot_sync(0xffffffffu, g <= tauE - Eh);
        while (hits) {
            const int src = __ffs(hits) - 1;
            hits &= hits - 1;
            if (lane == src) {
#pragma unroll
                for (int x = 0; x < NLO; ++x) scratch[x] = V[x];
#pragma unroll
                for (int x = 0; x < NMID; ++x) scratch[NLO + x] = U[x];
            }
            __syncwarp();
            const int eh = __shfl_sync(0xffffffffu, Eh, src);
            const unsigned long long qs = q0_warp + ((unsigned long long)src << nlow)
                                        + ((unsigned long long)(t ^ (t >> 1)) << LOWBITS) + (unsigned)lane;
            const int v = scratch[lane] + eh;
            for (int mid = 0; mid < NMID; ++mid) {
                const int e = v + sC[mid * NLO + lane] + scratch[NLO + mid];
                const unsigned long long q = qs + ((unsigned)mid << LL);
                if (e < tauE || (e == tauE && q < tauQ)) push_candidate(ctrl, pool, e, q);
            }
            __syncwarp();
        }
    }
}

// Direct evaluation of eq. (1) on the grid for `count` consecutive states starting at `base`; every state goes to the
// pool behind the `kept` entries already there. Used for the whole space when N <= N_DIRECT_MAX (2^N <= 16384 states)
// and for the first 2^15 states of any larger run (a2': with tau = +inf everything passes anyway, and one thread per
// state is the fastest way to form them).
__global__ void direct_kernel(const Tables* __restrict__ tab, Ctrl* __restrict__ ctrl, Entry* __restrict__ pool, int N,
                              unsigned long long base, unsigned count, unsigned kept)
{
    for (unsigned t = blockIdx.x * blockDim.x + threadIdx.x; t < count; t += gridDim.x * blockDim.x) {
        const unsigned long long q = base + t;
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
        pool[kept + t] = en;
    }
    if (blockIdx.x == 0 && threadIdx.x == 0) ctrl->count = kept + count;
}

void launch_enumerate(const Tables* tab, Ctrl* ctrl, Entry* pool, int N, int Lw,
                      unsigned long long base, unsigned nthreads, cudaStream_t st)
{
    const unsigned threads = nthreads < (unsigned)ENUM_THREADS ? nthreads : (unsigned)ENUM_THREADS;
    const unsigned blocks = (nthreads + threads - 1) / threads;
    enumerate_kernel<<<blocks, threads, 0, st>>>(tab, ctrl, pool, N, Lw, base, nthreads);
}

void launch_direct(const Tables* tab, Ctrl* ctrl, Entry* pool, int N, unsigned long long base, unsigned count,
                   unsigned kept, cudaStream_t st)
{
    const unsigned threads = 128, blocks = (count + threads - 1) / threads;
    direct_kernel<<<blocks, threads, 0, st>>>(tab, ctrl, pool, N, base, count, kept);
}

}  // namespace ising
