/*
 * ising.h -- C ABI of the B200-native exhaustive Ising enumerator
 *            (hot path of arXiv 1904.03621, "Brute-forcing spin-glass problems with CUDA").
 *
 * What the library computes (PAPER.md:9 abstract, eq. (1), Algorithm 1):
 * over all 2^N spin configurations of
 *
 *      H(s) = - sum_{i<j} J_ij s_i s_j - sum_i h_i s_i ,        s_i = +-1          (eq. 1)
 *
 * the S lowest (H, q) pairs, ascending under the total order (energy, state index).
 * State encoding (eqs. (4),(5); PAPER.md:58 q = (s+1)/2):
 * bit i of the 64-bit index q (bit 0 = least significant) is spin i; bit value 0 <-> s_i = -1,
 * bit value 1 <-> s_i = +1. Spin i is row/column i of J and entry i of h (0-based).
 *
 * All work runs in hand-written sm_100a CUDA kernels enqueued on the caller's stream. There is
 * no CPU fallback: without a CUDA device every compute entry point returns ISING_ERR_CUDA.
 * Every configuration of the requested range is screened against the running S-th best energy --
 * in blocks of 2^14 by a bf16 tensor-core (tcgen05) partition-function bound for the bulk of ranges
 * of 2^36 states and more, in blocks of 2^10 by a packed 16-bit lower bound otherwise -- and every
 * block that passes a screen is formed exactly in 32-bit integers; both screens can only add work
 * (false hits), never lose a state (DESIGN.md sections 6, 6b). Environment knobs (development /
 * tests): ISING_KERNEL = 16 (packed screen only) | 32 (int32 add-min per configuration, no screen),
 * ISING_Z_MIN_LOG2, ISING_Z_RAMP_LOG2, ISING_Z_FORCE = 1 (the bulk takes the tensor-core screen whatever its probe
 * flagged), ISING_LW, ISING_CHUNK_LOG2, ISING_GROWTH, ISING_PATH = 1
 * (host-sequenced pieces), ISING_KEEP_CAP_LOG2.
 *
 * Pointer arguments say in their name where they live: *_dev = device memory, *_host = host memory.
 * The library never frees or retains caller buffers. Scratch (two 64 MiB candidate pools, a 257 KiB
 * candidate histogram, the instance tables, a pinned control block) is allocated on first use per host
 * thread and device, reused by that thread's later calls, and released by ising_release_workspace()
 * or when the thread exits.
 * Every compute entry point SYNCHRONISES the stream before it returns (normally once, at the end: the
 * threshold is refreshed on the device), so outputs are valid on return. On any error the output buffers are left untouched
 * (device variants) or unspecified (host variants) and a negative ISING_ERR_* code is returned.
 * Nothing throws across this boundary. Calls on different streams may run concurrently.
 */
#ifndef ISING_H_
#define ISING_H_

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#define ISING_OK               0
#define ISING_ERR_NULL        -1   /* a required pointer is NULL */
#define ISING_ERR_BAD_N       -2   /* N < 1 or N > ISING_N_MAX */
#define ISING_ERR_BAD_S       -3   /* S < 1, S > number of states in the range, or S > ISING_S_MAX */
#define ISING_ERR_NONFINITE   -4   /* NaN or Inf in J or h */
#define ISING_ERR_ASYMMETRIC  -5   /* J[i*N+j] != J[j*N+i] */
#define ISING_ERR_DIAGONAL    -6   /* J[i*N+i] != 0 (fields go in h, not on the diagonal) */
#define ISING_ERR_BAD_RANGE   -7   /* q_begin >= q_end, q_end > 2^N, or bounds not multiples of 2^min(N,20) */
#define ISING_ERR_CUDA        -8   /* a CUDA runtime call failed; see ising_last_error() */
#define ISING_ERR_BAND        -9   /* guard band could not certify the result */
#define ISING_ERR_INTERNAL   -10
#define ISING_ERR_RANGE_W    -11   /* sum|J|+sum|h| is zero-scaled or too large/small to quantise */

#define ISING_N_MAX   63
#define ISING_S_MAX   65536

/*
 * ising_lowest -- the S lowest-energy states of the whole configuration space.
 * (BASELINE.json north_star signature; Algorithm 1 is the paper's version of the same job.)
 *
 *   J_dev            [N*N] float64, row-major, symmetric, zero diagonal; edge {i,j} has coupling J[i*N+j]
 *   h_dev            [N]   float64 fields
 *   N                number of spins, 1 <= N <= ISING_N_MAX
 *   S                number of states wanted, 1 <= S <= min(2^N, ISING_S_MAX)
 *   states_out_dev   [S] uint64  state indices q, ascending by (energy, q)
 *   energies_out_dev [S] float64 eq. (1) energies of those states, evaluated in fp64 in the fixed
 *                    order "pairs i<j row-major, then fields" (integer-valued inputs give exact integers)
 *   stream           a cudaStream_t passed as void* (NULL = default stream)
 *
 * Integer-valued (more generally: dyadic, exactly representable on the internal 2^-p grid) instances
 * are enumerated exactly and the result is bit-exact. Other real-valued instances are enumerated on a
 * fixed-point grid with a rigorous guard band and re-evaluated in fp64. If more
 * than 2^20 states lie inside the band of the S-th level (huge levels of states that tie on the grid), a
 * second enumeration streams exactly those states through the fp64 re-evaluation (ising_stats.passes = 2);
 * ISING_ERR_BAND is reserved and not returned by the current paths.
 */
int ising_lowest(const double *J_dev, const double *h_dev, int N, int S,
                 uint64_t *states_out_dev, double *energies_out_dev, void *stream);

/*
 * ising_lowest_range -- same, restricted to states q_begin <= q < q_end.
 * Both bounds must be multiples of 2^min(N,20) (so for N <= 20 only the full range is legal).
 * This is the unit of multi-GPU sharding, time slicing and checkpoint/resume (PAPER.md:85 chunks, eq. (6)).
 */
int ising_lowest_range(const double *J_dev, const double *h_dev, int N, int S,
                       uint64_t q_begin, uint64_t q_end,
                       uint64_t *states_out_dev, double *energies_out_dev, void *stream);

/*
 * ising_lowest_host -- end-to-end convenience: HOST buffers in, HOST buffers out. Copies J and h to
 * the device, runs ising_lowest_range on `stream`, copies the S results back. Same semantics and codes.
 */
int ising_lowest_host(const double *J_host, const double *h_host, int N, int S,
                      uint64_t q_begin, uint64_t q_end,
                      uint64_t *states_out_host, double *energies_out_host, void *stream);

/*
 * ising_merge_lists -- the exchange step of range sharding ("low_en/low_st" merge).
 * Input: n (state, energy) pairs (e.g. the concatenated per-range results); output: the S lowest under
 * (energy, q), ascending. 1 <= S <= n. Duplicated states are NOT removed (ranges are disjoint).
 */
int ising_merge_lists(const uint64_t *states_in_dev, const double *energies_in_dev, int64_t n, int S,
                      uint64_t *states_out_dev, double *energies_out_dev, void *stream);

/*
 * ising_merge_lists_static -- ising_merge_lists for callers that cannot allocate device memory. Same operation
 * (PAPER.md:103-110), same arguments, same result bit for bit, for n <= ISING_MERGE_STATIC_MAX.
 *
 * Why it exists: every other compute entry point creates, on a host thread's first call, a workspace of about
 * 130 MiB with cudaMalloc. A caller cannot do that when the device's memory already belongs, all of it, to another
 * allocator in the same process (a framework that reserves the GPU at start-up), and does not want to when the
 * device-wide synchronisation inside cudaMalloc / cudaFree would stall its other streams, or when the thread does
 * nothing but merge the per-range lists of a sharded run. This entry point calls no cudaMalloc, cudaFree,
 * cudaMallocHost or allocating library routine, ever: its sort scratch is a fixed 2 MiB array inside the library
 * image (ISING_MERGE_STATIC_MAX entries of 16 bytes), resident on every GPU that loads the library until the process
 * ends. Inputs and outputs remain the caller's buffers.
 *
 *   n > ISING_MERGE_STATIC_MAX          ISING_ERR_BAD_S, ising_last_error() names the limit; nothing is launched
 *   first call on a device              also looks up the array's device address and sets a kernel attribute:
 *                                       make it before any stream capture begins on that device
 *   calls that overlap on the GPU       share the one array and RACE (wrong results, no error): serialise calls
 *                                       per device. Back-to-back calls are fine: the array keeps the last call's
 *                                       entries, but each call overwrites or pads every slot it later reads.
 * Synchronises `stream` before returning, like ising_merge_lists.
 */
#define ISING_MERGE_STATIC_MAX 131072
int ising_merge_lists_static(const uint64_t *states_in_dev, const double *energies_in_dev, int64_t n, int S,
                             uint64_t *states_out_dev, double *energies_out_dev, void *stream);

/*
 * ising_dos -- density of states (cf. the paper's Fig. 6): the histogram
 * of ALL 2^N energies of eq. (1). Every energy is formed exactly on the library's 2^-p grid (the instance rounded to
 * multiples of 2^-p; for integer / dyadic instances that is the instance itself, otherwise each energy is within
 * ising_stats.epsilon of eq. (1)) and counted:
 *      hist_out_dev[b] = #{ q : e_lo + b * width <= E_grid(q) < e_lo + (b + 1) * width },   0 <= b < nbins
 * with e_lo = -(sum of |grid weights|) and width the smallest power-of-two multiple of 2^-p for which nbins bins
 * cover [-sum, +sum]; both are written to the two host doubles. 2 <= nbins <= 4096. sum_b hist[b] = 2^N.
 * J_dev, h_dev as in ising_lowest; hist_out_dev [nbins] uint64 device memory. Bound by shared-memory atomics
 * (about 10^12 states/s), not the hot path.
 */
int ising_dos(const double *J_dev, const double *h_dev, int N, int nbins, uint64_t *hist_out_dev,
              double *e_lo_out_host, double *bin_width_out_host, void *stream);

/*
 * ising_lowest_alg1 -- the PAPER'S OWN pipeline (Algorithm 1), written plainly for this GPU, as the
 * on-box comparison for the design above: the range is cut into chunks of
 * 2^chunk_log2 states (10 <= chunk_log2 <= 20); every state's energy is evaluated directly by eq. (1) in fp64,
 * O(N^2) per state, the chunk is stored in device memory behind the S lowest found so far
 * (low_en / low_st) and the S lowest of the two are selected by a full sort. No Gray walk, no
 * tables, no threshold filter, no grid or guard band: an independent exact path, several thousand times slower.
 * Same arguments, result, order and error codes as ising_lowest_range.
 */
int ising_lowest_alg1(const double *J_dev, const double *h_dev, int N, int S, uint64_t q_begin, uint64_t q_end,
                      int chunk_log2, uint64_t *states_out_dev, double *energies_out_dev, void *stream);

/*
 * ising_lowest_h0 -- zero-field instances (h = 0), using the global spin-flip symmetry E(q) = E(~q) of eq. (1)
 * (SURVEY.md section 8(f) item 3): only the half space q < 2^(N-1) is enumerated, every kept state brings its
 * complement (same fp64 energy) with it, and the 2 S candidates are ordered by (energy, q) and cut at S.
 * The result equals ising_lowest(J, 0, N, S) element for element; ising_stats.configs reports the 2^(N-1)
 * configurations actually evaluated (half the space: an EFFECTIVE rate must not be quoted as configs/s evaluated).
 * For N <= 20 the whole space is enumerated. J_dev as in ising_lowest.
 */
int ising_lowest_h0(const double *J_dev, int N, int S, uint64_t *states_out_dev, double *energies_out_dev, void *stream);

/*
 * qubo_lowest -- QUBO entry point, eqs. (2),(3):
 *      F(q) = - sum_{i<j} a_ij q_i q_j - sum_i b_i q_i ,   q_i in {0,1}
 * a_dev [N*N] symmetric zero-diagonal, b_dev [N]. Converted on the device to the equivalent Ising
 * instance (J = a/4, h_i = b_i/2 + sum_j a_ij/4, offset = -sum_i b_i/2 - sum_{i<j} a_ij/4) and
 * enumerated by the same kernels; energies_out holds F(q) evaluated directly in fp64.
 */
int qubo_lowest(const double *a_dev, const double *b_dev, int N, int S,
                uint64_t *states_out_dev, double *energies_out_dev, void *stream);

/*
 * ising_energies -- eq. (1) in fp64 for a list of n states (the re-evaluation kernel on its own).
 */
int ising_energies(const double *J_dev, const double *h_dev, int N,
                   const uint64_t *states_dev, int64_t n, double *energies_out_dev, void *stream);

/*
 * Statistics of the last successful compute call made by the calling thread (for bench.py / tests).
 * All counters refer to that one call.
 */
typedef struct ising_stats {
    uint64_t configs;            /* configurations whose energy was computed (= q_end - q_begin per pass) */
    uint64_t candidates;         /* (E, q) pairs that passed the threshold filter and reached a merge */
    uint32_t kernel_launches;    /* kernels of this library launched */
    uint32_t enum_launches;      /* of which enumeration kernels */
    uint32_t passes;             /* enumerations of the range: 1; +1 if the single pass overflowed the candidate pool and
                                    was redone piecewise; +1 for the band pass (more than 2^20 states within the guard band) */
    uint32_t split_retries;      /* launches re-run in halves after a candidate-buffer overflow */
    int32_t  grid_exponent;      /* p: weights were quantised to multiples of 2^-p */
    int32_t  exact;              /* 1 if the grid represents every weight exactly (integer / dyadic instance) */
    double   epsilon;            /* rigorous bound on |grid energy - true energy| (0 if exact) */
    double   enum_ms;            /* device time spent in enumeration kernels (CUDA events) */
    double   total_ms;           /* device time of the whole call */
    int32_t  keep;               /* K: candidates kept per list */
    int32_t  inner_bits;         /* L: unrolled Gray bits per inner block */
    int32_t  kernel_variant;     /* 1: ising_lowest_alg1. 2: ising_dos. 16: packed 16-bit screen + exact int32 re-forming of hit blocks;
                                    32: int32 add-min per configuration (environment ISING_KERNEL=32);
                                    128: as 16 for the ramp-up, the bulk through the tensor-core (tcgen05) screen (default
                                    for ranges of 2^36 states and more) */
    int32_t  screen_shift;       /* variant 16: one 16-bit unit = 2^screen_shift grid units (0: screen is exact) */
    uint64_t hit_blocks;         /* 1024-configuration blocks that passed the screen and were formed exactly (int32) */
    uint64_t false_hit_blocks;   /* ... of which none held a candidate (the price of the 16-bit screen; 0 for variant 32) */
    /* tensor-core screen (variant 128 only, else 0) */
    double   z_ms;               /* device time of the launches of the tensor-core screen kernel (part of enum_ms) */
    uint64_t z_configs;          /* configurations those launches covered (probe + bulk) */
    uint64_t z_blocks;           /* 2^14-configuration blocks screened by one row of a 128 x 128 x 128 GEMM each */
    uint64_t z_flagged_blocks;   /* ... of which flagged and formed exactly (16 blocks of 1024 each, counted in hit_blocks) */
    uint32_t z_launches;         /* launches of the tensor-core screen kernel (part of enum_launches) */
    uint32_t reserved0;
} ising_stats;

int ising_get_last_stats(ising_stats *out_host);

const char *ising_strerror(int status);
const char *ising_last_error(void);   /* thread-local detail string of the last failure */
int ising_version(void);

/* FP32-FMA microbenchmark (denominator of BASELINE.json's "FP32 FMA roofline" yardstick, bench.py `fp32_fma_roofline`):
 * runs a dependency-free FFMA kernel for roughly `ms_target` milliseconds on `stream` and writes the measured FMA/s
 * (lane-FMAs per second, whole GPU). */
int ising_fma_peak(double ms_target, double *fma_per_s_out_host, void *stream);

/* Same for the enumeration's inner operation, one fused integer add-min (SASS VIADDMNMX) per configuration:
 * lane add-mins per second, whole GPU. This is the ALU ceiling bench.py's `roofline_int32` (the int32 kernel, ISING_KERNEL=32) is
 * quoted against; the default path's `roofline` is a tensor-core roofline. */
int ising_addmin_peak(double ms_target, double *addmin_per_s_out_host, void *stream);

/* Same for the packed inner operation of the packed-screen kernel (SASS VIADDMNMX.U16x2): lane INSTRUCTIONS per second,
 * whole GPU; each instruction forms two 16-bit add-mins, i.e. screens two configurations, so the configuration
 * ceiling of the packed kernel is twice this number. */
int ising_addmin16x2_peak(double ms_target, double *inst_per_s_out_host, void *stream);

/* The instruction MIX the packed-screen kernel (walk_kernel<Inner16>) is built from, register-only: per chain step one fused VIADDMNMX.U16x2
 * (two 16-bit add-mins, ALU pipe) and one split group IMAD + IMAD + VIMNMX3.U16x2 (four add-mins: two packed sums on
 * the FMA pipe, one three-way packed minimum on the ALU pipe). Writes lane ADD-MINS per second, whole GPU: the
 * measured counterpart of the derived bound of DESIGN.md 5.2 (192 add-mins per clock per SM) and the denominator of
 * bench.py's `roofline_packed16.peak`. */
int ising_addmin_mix_peak(double ms_target, double *addmin_per_s_out_host, void *stream);

/* Self-test of the hardware property the tensor-core screen's proof relies on (csrc/zscreen.cu): one
 * 128 x 128 x 128 bf16 tcgen05 GEMM of pseudo-random POSITIVE operands spanning 2^-100 .. 2^40, fp32 accumulation in
 * tensor memory, compared entry by entry with the same sums formed in fp64 from the same bf16 values. Writes the
 * largest relative UNDER-estimate (ref - D) / ref and over-estimate (D - ref) / ref. The screen's margin (0.05 bits,
 * i.e. 3.5 %) budgets 2^-14 for this term. */
int ising_zscreen_selftest(uint32_t seed, double *rel_under_out_host, double *rel_over_out_host, void *stream);

/* Frees the calling thread's cached workspace (device pool, tables, pinned control block). Optional. */
void ising_release_workspace(void);

#ifdef __cplusplus
}
#endif
#endif /* ISING_H_ */
