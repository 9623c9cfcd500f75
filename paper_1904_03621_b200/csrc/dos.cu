// dos.cu -- density-of-states mode (the paper's Fig. 6 compares densities of states,
// PAPER.md:229): every one of the 2^N grid energies is formed exactly (int32, same tables and Gray walk as
// enumerate.cu) and counted in a histogram instead of being compared with a threshold.
//
//   E(q) = Eh + U[mid] + V[lo] + C[mid][lo]      (the QUBO decomposition of eqs. (2),(3))
//   bin  = (E - e_lo) >> bshift                  (bins of 2^bshift grid units, i.e. 2^(bshift - p) in energy)
//
// Counting: one shared-memory histogram per block (32-bit counters; a block forms at most 2^28 energies), updated
// with shared atomics, flushed to the 64-bit global histogram when the block ends. This mode is bound by the shared
// atomic unit, not by the ALU pipe; it is a side feature, not the hot path.
#include "common.cuh"

namespace ising {

constexpr int DOS_THREADS = 256;
constexpr int DOS_MAX_BINS = 4096;

__global__ void __launch_bounds__(DOS_THREADS, 2)
dos_kernel(const Tables* __restrict__ tab, int N, int Lw, unsigned long long base, unsigned nthreads,
           int e_lo, int bshift, int nbins, unsigned long long* __restrict__ hist)
{
    __shared__ __align__(16) int sC[NMID * NLO];
    __shared__ __align__(16) int sDV[LW_MAX * 2 * NLO];
    __shared__ __align__(16) int sDU[LW_MAX * 2 * NMID];
    __shared__ int sDW[1 << LW_MAX];
    __shared__ unsigned sHist[DOS_MAX_BINS];

    for (int i = threadIdx.x; i < NMID * NLO; i += blockDim.x) sC[i] = tab->C[i];
    for (int i = threadIdx.x; i < LW_MAX * 2 * NLO; i += blockDim.x) sDV[i] = tab->DV[i];
    for (int i = threadIdx.x; i < LW_MAX * 2 * NMID; i += blockDim.x) sDU[i] = tab->DU[i];
    for (int i = threadIdx.x; i < (1 << Lw); i += blockDim.x) sDW[i] = tab->DW[i];
    for (int i = threadIdx.x; i < nbins; i += blockDim.x) sHist[i] = 0u;
    __syncthreads();

    const unsigned gtid = blockIdx.x * blockDim.x + threadIdx.x;
    if (gtid < nthreads) {
        const int nlow = LOWBITS + Lw;
        const unsigned long long q0 = base + ((unsigned long long)gtid << nlow);
        const int* __restrict__ Jq = tab->Jq;
        const int* __restrict__ hq = tab->hq;
        // base state: E(q0) by eq. (1) and the local fields of the lo, mid and walk spins
        int E0 = 0;
        for (int i = 0; i < N; ++i) {
            const unsigned bi = (unsigned)(q0 >> i) & 1u;
            const int* row = Jq + i * 64;
            int acc = 0;
            for (int j = i + 1; j < N; ++j) {
                const int v = row[j];
                acc += (bi ^ ((unsigned)(q0 >> j) & 1u)) ? v : -v;
            }
            const int hv = hq[i];
            E0 += acc + (bi ? -hv : hv);
        }
        int Phi[LOWBITS + LW_MAX];
#pragma unroll
        for (int i = 0; i < LOWBITS + LW_MAX; ++i) {
            int acc = 0;
            if (i < nlow && i < N) {
                const int* row = Jq + i * 64;
                acc = hq[i];
                for (int j = 0; j < N; ++j) {
                    const int v = row[j];
                    acc += ((unsigned)(q0 >> j) & 1u) ? v : -v;
                }
            }
            Phi[i] = acc;
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
        int Eh = E0 - e_lo;                       // energies relative to the lower edge of bin 0

        const unsigned nsteps = 1u << Lw;
        for (unsigned t = 0; t < nsteps; ++t) {
            if (t > 0) {
                const int k = __ffs(t) - 1;
                const unsigned gnew = t ^ (t >> 1);
                const int sb = (gnew >> k) & 1;
                int phi = Phi[LOWBITS];
#pragma unroll
                for (int kk = 1; kk < LW_MAX; ++kk) phi = (k == kk) ? Phi[LOWBITS + kk] : phi;
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
#pragma unroll
            for (int mid = 0; mid < NMID; ++mid) {
                const int off = U[mid] + Eh;
                const int4* crow = reinterpret_cast<const int4*>(sC + mid * NLO);
#pragma unroll
                for (int x = 0; x < NLO / 4; ++x) {
                    const int4 c = crow[x];
                    atomicAdd(&sHist[(unsigned)(V[4 * x + 0] + c.x + off) >> bshift], 1u);
                    atomicAdd(&sHist[(unsigned)(V[4 * x + 1] + c.y + off) >> bshift], 1u);
                    atomicAdd(&sHist[(unsigned)(V[4 * x + 2] + c.z + off) >> bshift], 1u);
                    atomicAdd(&sHist[(unsigned)(V[4 * x + 3] + c.w + off) >> bshift], 1u);
                }
            }
        }
    }
    __syncthreads();
    for (int i = threadIdx.x; i < nbins; i += blockDim.x) {
        const unsigned c = sHist[i];
        if (c) atomicAdd(&hist[i], (unsigned long long)c);
    }
}

void launch_dos(const Tables* tab, int N, int Lw, unsigned long long base, unsigned nthreads, int e_lo, int bshift,
                int nbins, unsigned long long* hist, cudaStream_t st)
{
    const unsigned threads = nthreads < (unsigned)DOS_THREADS ? nthreads : (unsigned)DOS_THREADS;
    const unsigned blocks = (nthreads + threads - 1) / threads;
    dos_kernel<<<blocks, threads, 0, st>>>(tab, N, Lw, base, nthreads, e_lo, bshift, nbins, hist);
}

// N <= N_DIRECT_MAX: one thread per state, eq. (1) on the grid, global 64-bit atomics
__global__ void dos_direct_kernel(const Tables* __restrict__ tab, int N, int e_lo, int bshift,
                                  unsigned long long* __restrict__ hist)
{
    const unsigned total = 1u << N;
    for (unsigned q = blockIdx.x * blockDim.x + threadIdx.x; q < total; q += gridDim.x * blockDim.x) {
        int e = 0;
        for (int i = 0; i < N; ++i) {
            const unsigned bi = (q >> i) & 1u;
            for (int j = i + 1; j < N; ++j) {
                const int v = tab->Jq[i * 64 + j];
                e += (bi ^ ((q >> j) & 1u)) ? v : -v;
            }
            const int hv = tab->hq[i];
            e += bi ? -hv : hv;
        }
        atomicAdd(&hist[(unsigned)(e - e_lo) >> bshift], 1ull);
    }
}

void launch_dos_direct(const Tables* tab, int N, int e_lo, int bshift, unsigned long long* hist, cudaStream_t st)
{
    const unsigned total = 1u << N;
    dos_direct_kernel<<<(total + 127) / 128, 128, 0, st>>>(tab, N, e_lo, bshift, hist);
}

}  // namespace ising
