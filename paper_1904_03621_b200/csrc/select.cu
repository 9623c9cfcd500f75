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
            Entry e = s[i];
            const bool asc = ((gbase + i) & k) == 0;
            for (int jj = j; jj >= 1; jj >>= 1) {
                const bool lower = (i & jj) == 0;
                e = shfl_exchange(e, jj, lower == asc);
            }
            s[i] = e;
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

// After the sort: how many entries stay, and the new threshold (a5/a6 "publish the K-th best").
__global__ void truncate_kernel(const Entry* __restrict__ pool, Ctrl* __restrict__ ctrl, unsigned n, int S)
{
    if (threadIdx.x != 0 || blockIdx.x != 0) return;
    unsigned keep = n;
    int tauE = TAU_INF;
    unsigned long long tauQ = Q_MAX;
    if (n >= (unsigned)S) {
        const int eS = i32_from_key(pool[S - 1].key);
        if (ctrl->exact) {
            keep = (unsigned)S;
            tauE = eS;
            tauQ = pool[S - 1].q;
        } else {
            tauE = eS + ctrl->band;
            const unsigned long long kmax = key_from_i32(tauE);
            unsigned lo = (unsigned)S, hi = n;           // first index in [S, n) with key > kmax
            while (lo < hi) {
                const unsigned mid = (lo + hi) >> 1;
                if (pool[mid].key <= kmax) lo = mid + 1; else hi = mid;
            }
            keep = lo;
        }
    }
    if (keep > KEEP_CAP) { keep = KEEP_CAP; ctrl->band_overflow = 1; }
    ctrl->kept = keep;
    ctrl->count = keep;
    ctrl->tauE = tauE;
    ctrl->tauQ = tauQ;
}

static unsigned long long next_pow2(unsigned long long x)
{
    unsigned long long p = 1;
    while (p < x) p <<= 1;
    return p;
}

static bool g_smem_attr_set = false;

// Sort pool[0..n) ascending by (key, q); entries in [n, P) are sentinels afterwards. Returns kernels launched.
static int sort_pool(Entry* pool, unsigned n, cudaStream_t st)
{
    if (!g_smem_attr_set) {
        cudaFuncSetAttribute(tile_sort_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, SORT_TILE * (int)sizeof(Entry));
        cudaFuncSetAttribute(tile_merge_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, SORT_TILE * (int)sizeof(Entry));
        g_smem_attr_set = true;
    }
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

int launch_select(Entry* pool, Ctrl* ctrl, unsigned n, int S, cudaStream_t st)
{
    int launches = sort_pool(pool, n, st);
    truncate_kernel<<<1, 32, 0, st>>>(pool, ctrl, n, S);
    return launches + 1;
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
            acc += -si * h[i];
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

}  // namespace ising
