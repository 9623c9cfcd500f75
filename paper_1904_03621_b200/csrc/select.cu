// select.cu -- SURVEY.md section 8 rows a5 (block top-K with bitonic networks), a6 (merge) and a7 (exact fp64
// re-evaluation, final order, output). The paper's counterpart is select_lowest on low_en/low_st[2 num_st] and the
// final sort_by_key (Algorithm 1).
//
// The pool is ONE array: a sorted prefix of `kept` entries (the best so far) followed by the candidates the
// enumeration pushed since. A selection sorts pool[0..n) by (key, q) with a bitonic network -- one block in shared
// memory when n <= SORT_TILE (the common case), tile sorts plus global merge steps otherwise -- and then truncates:
// exact instances keep S entries, others keep everything within the guard band of the S-th.
#include "common.cuh"

namespace ising {

__device__ __forceinline__ void cmp_swap(Entry& a, Entry& b, bool ascending)
{
    const bool sw = ascending ? entry_less(b, a) : entry_less(a, b);
    if (sw) { Entry t = a; a = b; b = t; }
}

// Exchange with the lane `lane ^ j` (j < 32): each lane keeps the smaller or the larger of the pair.
// This is the warp-shuffle leg of the bitonic network (north_star (c)).
__device__ __forceinline__ Entry shfl_exchange(const Entry& mine, int j, bool keep_small)
{
    Entry o;
    o.key = __shfl_xor_sync(0xffffffffu, mine.key, j);
    o.q = __shfl_xor_sync(0xffffffffu, mine.q, j);
    const bool other_less = entry_less(o, mine);
    return (other_less == keep_small) ? o : mine;
}

// Bitonic stages j = jstart .. 1 of merge size k on a tile held in shared memory. `gbase` is the tile's global index
// offset (the sort direction of a pair depends on the global index). Strides j >= 32 go through shared memory,
// strides j < 32 through warp shuffles with one element per lane (tile processed in slices of blockDim entries).
__device__ void tile_stages(Entry* s, int tile, unsigned long long gbase, unsigned long long k, int jstart)
{
    int j = jstart;
    for (; j >= 32; j >>= 1) {
        for (int i = threadIdx.x; i < tile / 2; i += blockDim.x) {
            const int l = 2 * i - (i & (j - 1));
            const bool asc = ((gbase + l) & k) == 0;
            cmp_swap(s[l], s[l + j], asc);
        }
        __syncthreads();
    }
    if (j >= 1) {
        for (int i0 = 0; i0 < tile; i0 += blockDim.x) {
            const int i = i0 + threadIdx.x;            // tile and blockDim are multiples of 32
            if (i < tile) {                            // warp-uniform (a block may be wider than a small tile)
                Entry e = s[i];
                const bool asc = ((gbase + i) & k) == 0;
                for (int jj = j; jj >= 1; jj >>= 1) {
                    const bool lower = (i & jj) == 0;
                    e = shfl_exchange(e, jj, lower == asc);
                }
                s[i] = e;
            }
        }
        __syncthreads();
    }
}

// Full bitonic sort of every SORT_TILE-sized tile (merge sizes k = 2 .. tile); n_fill: entries >= n become sentinels.
__global__ void __launch_bounds__(SORT_THREADS) tile_sort_kernel(Entry* __restrict__ pool, unsigned n, int tile)
{
    extern __shared__ __align__(16) unsigned char smem_raw[];
    Entry* s = reinterpret_cast<Entry*>(smem_raw);
    const unsigned long long gbase = (unsigned long long)blockIdx.x * tile;
    for (int i = threadIdx.x; i < tile; i += blockDim.x) {
        Entry e;
        if (gbase + i < n) e = pool[gbase + i];
        else { e.key = ~0ull; e.q = ~0ull; }
        s[i] = e;
    }
    __syncthreads();
    for (unsigned long long k = 2; k <= (unsigned long long)tile; k <<= 1)
        tile_stages(s, tile, gbase, k, (int)(k >> 1));
    for (int i = threadIdx.x; i < tile; i += blockDim.x) pool[gbase + i] = s[i];
}

// One global compare-exchange stage (stride j >= SORT_TILE) of merge size k.
__global__ void global_stage_kernel(Entry* __restrict__ pool, unsigned long long P, unsigned long long k,
                                    unsigned long long j)
{
    const unsigned long long i = (unsigned long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= P / 2) return;
    const unsigned long long l = 2 * i - (i & (j - 1));
    Entry a = pool[l], b = pool[l + j];
    const bool asc = (l & k) == 0;
    const bool sw = asc ? entry_less(b, a) : entry_less(a, b);
    if (sw) { pool[l] = b; pool[l + j] = a; }
}

// Stages j = tile/2 .. 1 of merge size k > tile, per tile in shared memory.
__global__ void __launch_bounds__(SORT_THREADS) tile_merge_kernel(Entry* __restrict__ pool, unsigned long long k, int tile)
{
    extern __shared__ __align__(16) unsigned char smem_raw[];
    Entry* s = reinterpret_cast<Entry*>(smem_raw);
    const unsigned long long gbase = (unsigned long long)blockIdx.x * tile;
    for (int i = threadIdx.x; i < tile; i += blockDim.x) s[i] = pool[gbase + i];
    __syncthreads();
    tile_stages(s, tile, gbase, k, tile >> 1);
    for (int i = threadIdx.x; i < tile; i += blockDim.x) pool[gbase + i] = s[i];
}

// How many entries of a sorted list stay, and the threshold they certify (a5/a6 "publish the K-th best"):
// exact instances keep S entries, others everything within the guard band of the S-th.
// Returns the number kept; tau_out = the threshold word, eS_out = the S-th smallest grid energy.
__device__ unsigned truncate_sorted(const Entry* pool, unsigned n, int S, int exact, int band,
                                    unsigned long long q_begin, int qshift, unsigned long long& tau_out, int& eS_out)
{
    unsigned keep = n;
    tau_out = tau_pack(TAU_INF, QC_NONE);
    eS_out = TAU_INF;
    if (n >= (unsigned)S) {
        const int eS = i32_from_key(pool[S - 1].key);
        eS_out = eS;
        if (exact) {
            keep = (unsigned)S;
            // ties on eS pass only below the S-th state's successor, rounded up to the coarse grid of the word
            const unsigned long long d = pool[S - 1].q + 1ull - q_begin;
            const unsigned long long v = (d + ((1ull << qshift) - 1ull)) >> qshift;
            tau_out = tau_pack(eS, v < (unsigned long long)QC_NONE ? (unsigned)v : QC_NONE);
        } else {
            const long long t = (long long)eS + band;
            const int tauE = t < (long long)TAU_INF ? (int)t : TAU_INF;
            tau_out = tau_pack(tauE, QC_NONE);
            const unsigned long long kmax = key_from_i32(tauE);
            unsigned lo = (unsigned)S, hi = n;           // first index in [S, n) with key > kmax
            while (lo < hi) {
                const unsigned mid = (lo + hi) >> 1;
                if (pool[mid].key <= kmax) lo = mid + 1; else hi = mid;
            }
            keep = lo;
        }
    }
    return keep;
}

// After the sort of a host-sequenced selection: truncate and publish.
__global__ void truncate_kernel(const Entry* __restrict__ pool, Ctrl* __restrict__ ctrl, unsigned n, int S,
                                unsigned long long q_begin, int qshift, unsigned keep_cap)
{
    if (threadIdx.x != 0 || blockIdx.x != 0) return;
    unsigned long long tau;
    int eS;
    unsigned keep = truncate_sorted(pool, n, S, ctrl->exact, ctrl->band, q_begin, qshift, tau, eS);
    if (keep > keep_cap) { keep = keep_cap; ctrl->band_overflow = 1; }
    ctrl->kept = keep;
    ctrl->count = keep;
    ctrl->eS = eS;
    atomicMin(&ctrl->tau, tau);
}

static unsigned long long next_pow2(unsigned long long x)
{
    unsigned long long p = 1;
    while (p < x) p <<= 1;
    return p;
}

// cudaFuncAttributeMaxDynamicSharedMemorySize is a per-DEVICE attribute: api.cu calls this whenever a host thread's
// workspace is (re)created on a device (cheap; no process-global flag).
void set_select_attributes();

// Sort pool[0..n) ascending by (key, q); entries in [n, P) are sentinels afterwards. Returns kernels launched.
static int sort_pool(Entry* pool, unsigned n, cudaStream_t st)
{
    int launches = 0;
    unsigned long long P = next_pow2(n < 32 ? 32 : n);
    if (P <= (unsigned long long)SORT_TILE) {
        const int tile = (int)P;
        const int threads = tile < SORT_THREADS ? tile : SORT_THREADS;
        tile_sort_kernel<<<1, threads, tile * sizeof(Entry), st>>>(pool, n, tile);
        return 1;
    }
    const int tile = SORT_TILE;
    const unsigned tiles = (unsigned)(P / tile);
    tile_sort_kernel<<<tiles, SORT_THREADS, tile * sizeof(Entry), st>>>(pool, n, tile);
    ++launches;
    for (unsigned long long k = 2ull * tile; k <= P; k <<= 1) {
        for (unsigned long long j = k >> 1; j >= (unsigned long long)tile; j >>= 1) {
            const unsigned blocks = (unsigned)((P / 2 + 255) / 256);
            global_stage_kernel<<<blocks, 256, 0, st>>>(pool, P, k, j);
            ++launches;
        }
        tile_merge_kernel<<<tiles, SORT_THREADS, tile * sizeof(Entry), st>>>(pool, k, tile);
        ++launches;
    }
    return launches;
}

int launch_select(Entry* pool, Ctrl* ctrl, unsigned n, int S, const Plan& plan, cudaStream_t st)
{
    int launches = sort_pool(pool, n, st);
    truncate_kernel<<<1, 32, 0, st>>>(pool, ctrl, n, S, plan.q_begin, plan.qshift, plan.keep_cap);
    return launches + 1;
}

// ---- single-pass path: drop every pool entry the final threshold excludes (a6, first half) ----
__global__ void __launch_bounds__(256) compact_kernel(const Entry* __restrict__ pool, Entry* __restrict__ pool2,
                                                      Ctrl* __restrict__ ctrl, unsigned long long q_begin, int qshift)
{
    if (ctrl->status != 0 || ctrl->pool_overflow) return;
    const unsigned n = ctrl->count < POOL_CAP ? ctrl->count : POOL_CAP;
    const unsigned long long tau = ctrl->tau;
    const unsigned long long kE = tau >> 32;
    const unsigned qc = tau_qc(tau);
    const unsigned long long tauQ = qc == QC_NONE ? Q_MAX : q_begin + ((unsigned long long)qc << qshift);
    const int lane = threadIdx.x & 31;
    const unsigned stride = gridDim.x * blockDim.x;
    for (unsigned i0 = blockIdx.x * blockDim.x; i0 < n; i0 += stride) {     // whole warps iterate together
        const unsigned i = i0 + threadIdx.x;
        Entry e;
        bool keep = false;
        if (i < n) {
            e = pool[i];
            keep = e.key < kE || (e.key == kE && e.q < tauQ);
        }
        const unsigned ball = __ballot_sync(0xffffffffu, keep);
        if (!ball) continue;
        unsigned base = 0;
        if (lane == 0) base = atomicAdd(&ctrl->count2, (unsigned)__popc(ball));
        base = __shfl_sync(0xffffffffu, base, 0);
        if (keep) pool2[base + __popc(ball & ((1u << lane) - 1u))] = e;
    }
}

int launch_compact(const Entry* pool, Entry* pool2, Ctrl* ctrl, const Plan& plan, cudaStream_t st)
{
    compact_kernel<<<296, 256, 0, st>>>(pool, pool2, ctrl, plan.q_begin, plan.qshift);
    return 1;
}

// ---- a7: eq. (1) (mode 0) or eq. (2) (mode 1: J holds a, h holds b) in fp64, fixed order: pairs i<j row-major, then fields ----
__device__ double energy_f64(const double* __restrict__ J, const double* __restrict__ h, int N, unsigned long long q, int mode)
{
    double acc = 0.0;
    if (mode == 0) {
        for (int i = 0; i < N; ++i) {
            const double si = (q >> i & 1ull) ? 1.0 : -1.0;
            for (int j = i + 1; j < N; ++j) {
                const double sj = (q >> j & 1ull) ? 1.0 : -1.0;
                acc += -(si * sj) * J[i * N + j];
            }
        }
        for (int i = 0; i < N; ++i) {
            const double si = (q >> i & 1ull) ? 1.0 : -1.0;
            acc += -si * (FIELD_TERM_SIGN * h[i]);
        }
    } else {
        for (int i = 0; i < N; ++i) {
            if (!(q >> i & 1ull)) continue;
            for (int j = i + 1; j < N; ++j)
                if (q >> j & 1ull) acc += -J[i * N + j];
        }
        for (int i = 0; i < N; ++i)
            if (q >> i & 1ull) acc += -h[i];
    }
    return acc;
}

__global__ void reeval_kernel(const double* __restrict__ J, const double* __restrict__ h, int N, int mode,
                              Entry* __restrict__ pool, unsigned m)
{
    const unsigned i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= m) return;
    pool[i].key = key_from_f64(energy_f64(J, h, N, pool[i].q, mode));
}

__global__ void emit_kernel(const Entry* __restrict__ pool, int S, unsigned long long* __restrict__ states_out,
                            double* __restrict__ energies_out)
{
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= S) return;
    states_out[i] = pool[i].q;
    energies_out[i] = f64_from_key(pool[i].key);
}

int launch_final(const double* J, const double* h, int N, int mode, Entry* pool, unsigned m, int S,
                 unsigned long long* states_out, double* energies_out, cudaStream_t st)
{
    reeval_kernel<<<(m + 127) / 128, 128, 0, st>>>(J, h, N, mode, pool, m);
    int launches = 1 + sort_pool(pool, m, st);
    emit_kernel<<<(S + 255) / 256, 256, 0, st>>>(pool, S, states_out, energies_out);
    return launches + 1;
}

__global__ void energies_kernel(const double* __restrict__ J, const double* __restrict__ h, int N, int mode,
                                const unsigned long long* __restrict__ states, long long n, double* __restrict__ out)
{
    const long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n) return;
    out[i] = energy_f64(J, h, N, states[i], mode);
}

void launch_energies(const double* J, const double* h, int N, int mode, const unsigned long long* states,
                     long long n, double* out, cudaStream_t st)
{
    if (n <= 0) return;
    energies_kernel<<<(unsigned)((n + 127) / 128), 128, 0, st>>>(J, h, N, mode, states, n, out);
}

__global__ void pack_kernel(const unsigned long long* __restrict__ states, const double* __restrict__ energies,
                            long long n, Entry* __restrict__ scratch)
{
    const long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n) return;
    Entry e;
    e.key = key_from_f64(energies[i]);
    e.q = states[i];
    scratch[i] = e;
}

// ---- the paper's own pipeline (Algorithm 1), written plainly: for comparison on the same box ----
// energies[j], states[j] of one chunk by direct evaluation of eq. (1) per state (O(N^2) each,
// PAPER.md:170), appended behind the `kept` lowest found so far (the paper's low_en / low_st).
__global__ void alg1_chunk_kernel(const double* __restrict__ J, const double* __restrict__ h, int N,
                                  unsigned long long base, unsigned count, Entry* __restrict__ dst)
{
    const unsigned i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= count) return;
    Entry e;
    e.q = base + i;
    e.key = key_from_f64(energy_f64(J, h, N, e.q, 0));
    dst[i] = e;
}

// One iteration of Algorithm 1: evaluate the chunk, then select_lowest over (kept + chunk) by a full sort.
int launch_alg1_chunk(const double* J, const double* h, int N, unsigned long long base, unsigned count,
                      Entry* pool, unsigned kept, cudaStream_t st)
{
    alg1_chunk_kernel<<<(count + 127) / 128, 128, 0, st>>>(J, h, N, base, count, pool + kept);
    return 1 + sort_pool(pool, kept + count, st);
}

int launch_emit(const Entry* pool, int S, unsigned long long* states_out, double* energies_out, cudaStream_t st)
{
    emit_kernel<<<(S + 255) / 256, 256, 0, st>>>(pool, S, states_out, energies_out);
    return 1;
}

// h = 0: E(q) = E(~q). Every kept state of the lower half space brings its complement (same energy) with it.
__global__ void expand_complement_kernel(const unsigned long long* __restrict__ states, const double* __restrict__ energies,
                                         int n, unsigned long long mask, Entry* __restrict__ scratch)
{
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n) return;
    Entry e;
    e.key = key_from_f64(energies[i]);
    e.q = states[i];
    scratch[2 * i] = e;
    e.q = ~states[i] & mask;
    scratch[2 * i + 1] = e;
}

int launch_expand_complements(const unsigned long long* states, const double* energies, int n, int N, int S,
                              Entry* scratch, unsigned long long* states_out, double* energies_out, cudaStream_t st)
{
    const unsigned long long mask = N >= 64 ? ~0ull : ((1ull << N) - 1ull);
    expand_complement_kernel<<<(n + 255) / 256, 256, 0, st>>>(states, energies, n, mask, scratch);
    int launches = 1 + sort_pool(scratch, 2u * (unsigned)n, st);
    emit_kernel<<<(S + 255) / 256, 256, 0, st>>>(scratch, S, states_out, energies_out);
    return launches + 1;
}

int launch_merge_lists(const unsigned long long* states, const double* energies, long long n, int S, Entry* scratch,
                       unsigned long long* states_out, double* energies_out, cudaStream_t st)
{
    pack_kernel<<<(unsigned)((n + 255) / 256), 256, 0, st>>>(states, energies, n, scratch);
    int launches = 1 + sort_pool(scratch, (unsigned)n, st);
    emit_kernel<<<(S + 255) / 256, 256, 0, st>>>(scratch, S, states_out, energies_out);
    return launches + 1;
}

// ---- single-pass path, a6 second half + a7 in ONE block: sort the compacted candidates by (grid energy, q), cut at
// the S-th (exact) or at the guard band (real weights), re-evaluate eq. (1) in fp64 in the oracle's summation order,
// sort by (E64, q), emit. Handles up to SORT_TILE candidates; more (large S) is left to the general kernels
// (Ctrl::final_state = 2). Writes nothing if the run was void (pool overflow) or the instance was rejected. ----
__global__ void __launch_bounds__(SORT_THREADS) final_small_kernel(const double* __restrict__ J, const double* __restrict__ h,
                                                                   int N, int mode, const Entry* __restrict__ pool2,
                                                                   Ctrl* __restrict__ ctrl, int S, unsigned keep_cap,
                                                                   unsigned long long* __restrict__ states_out,
                                                                   double* __restrict__ energies_out)
{
    extern __shared__ __align__(16) unsigned char smem_raw[];
    Entry* s = reinterpret_cast<Entry*>(smem_raw);
    __shared__ unsigned s_keep;
    if (ctrl->status != 0 || ctrl->pool_overflow) return;
    const unsigned n = ctrl->count2;
    if (n > (unsigned)SORT_TILE || n > keep_cap || n < (unsigned)S) {
        if (threadIdx.x == 0) ctrl->final_state = 2;
        return;
    }
    int tile = 32;
    while ((unsigned)tile < n) tile <<= 1;
    for (int i = threadIdx.x; i < tile; i += blockDim.x) {
        Entry e;
        if ((unsigned)i < n) e = pool2[i];
        else { e.key = ~0ull; e.q = ~0ull; }
        s[i] = e;
    }
    __syncthreads();
    for (unsigned long long k = 2; k <= (unsigned long long)tile; k <<= 1) tile_stages(s, tile, 0ull, k, (int)(k >> 1));
    if (threadIdx.x == 0) {
        unsigned long long tau;
        int eS;
        s_keep = truncate_sorted(s, n, S, ctrl->exact, ctrl->band, 0ull, 0, tau, eS);
        ctrl->kept = s_keep;
        ctrl->eS = eS;
    }
    __syncthreads();
    const unsigned keep = s_keep;
    int tile2 = 32;                                    // the kept entries are the first `keep` of the sorted tile
    while ((unsigned)tile2 < keep) tile2 <<= 1;
    for (int i = threadIdx.x; i < tile2; i += blockDim.x) {
        if ((unsigned)i < keep) s[i].key = key_from_f64(energy_f64(J, h, N, s[i].q, mode));
        else { s[i].key = ~0ull; s[i].q = ~0ull; }
    }
    __syncthreads();
    for (unsigned long long k = 2; k <= (unsigned long long)tile2; k <<= 1) tile_stages(s, tile2, 0ull, k, (int)(k >> 1));
    for (int i = threadIdx.x; i < S; i += blockDim.x) {
        states_out[i] = s[i].q;
        energies_out[i] = f64_from_key(s[i].key);
    }
    if (threadIdx.x == 0) ctrl->final_state = 1;
}

int launch_final_small(const double* J, const double* h, int N, int mode, Entry* pool2, Ctrl* ctrl, int S,
                       unsigned keep_cap, unsigned long long* states_out, double* energies_out, cudaStream_t st)
{
    final_small_kernel<<<1, SORT_THREADS, SORT_TILE * sizeof(Entry), st>>>(J, h, N, mode, pool2, ctrl, S, keep_cap,
                                                                            states_out, energies_out);
    return 1;
}

void set_select_attributes()
{
    cudaFuncSetAttribute(tile_sort_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, SORT_TILE * (int)sizeof(Entry));
    cudaFuncSetAttribute(tile_merge_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, SORT_TILE * (int)sizeof(Entry));
    cudaFuncSetAttribute(final_small_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, SORT_TILE * (int)sizeof(Entry));
}

// ---- band pass (the G3 fallback): pool[0..kept) holds the best `want` band states found so
// far, already keyed by their fp64 energy; pool[kept..n) holds new band states keyed by grid energy. Re-evaluate the
// new ones in fp64, sort everything by (E64, q), keep the lowest `want`. ----
__global__ void reeval_range_kernel(const double* __restrict__ J, const double* __restrict__ h, int N, int mode,
                                    Entry* __restrict__ pool, unsigned first, unsigned n)
{
    const unsigned i = first + blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n) return;
    pool[i].key = key_from_f64(energy_f64(J, h, N, pool[i].q, mode));
}
__global__ void set_count_kernel(Ctrl* ctrl, unsigned kept)
{
    ctrl->kept = kept;
    ctrl->count = kept;
}

int launch_band_drain(const double* J, const double* h, int N, int mode, Entry* pool, Ctrl* ctrl, unsigned kept,
                      unsigned n, unsigned want, cudaStream_t st)
{
    int launches = 0;
    if (n > kept) {
        reeval_range_kernel<<<(n - kept + 127) / 128, 128, 0, st>>>(J, h, N, mode, pool, kept, n);
        launches += 1 + sort_pool(pool, n, st);
    }
    set_count_kernel<<<1, 1, 0, st>>>(ctrl, n < want ? n : want);
    return launches + 1;
}

}  // namespace ising
