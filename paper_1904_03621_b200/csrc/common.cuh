// common.cuh -- shared declarations of the sm_100a CUDA path (product code; the CPU oracle shares nothing with it).
//
// Vocabulary:
//   spin i <-> bit i of q (bit 0 = LSB); bit value 0 <-> s_i = -1, 1 <-> s_i = +1
//   L  = "lo"   spins 0..LL-1          : per-thread register table V[2^LL]
//   M  = "mid"  spins LL..LL+LM-1      : per-thread register table U[2^LM], shared table C[2^LM][2^LL]
//   W  = "walk" spins LL+LM..+Lw-1     : walked by every thread in reflected Gray order
//   T  = "thread" spins above          : lane bits and the bits of the work unit; fixed per thread
//   all energies in the kernels are int32 multiples of the grid 2^-p (stage.cu chooses p).
//
// Work distribution: the state range of a call is cut into SEGMENTS of geometrically
// growing size; a segment is cut into equal UNITS (one warp each: 32 lanes x 2^Lw Gray steps x 1024 configurations,
// or, for the very first segment, one 1024-configuration block formed exactly). The persistent enumeration kernel
// hands units out in ascending order of q through an atomic counter in Ctrl.
#pragma once
#include <cstdint>
#include <cuda_runtime.h>

namespace ising {

constexpr int LL = 5;                    // lo bits
constexpr int LM = 5;                    // mid bits
constexpr int NLO = 1 << LL;
constexpr int NMID = 1 << LM;
constexpr int LOWBITS = LL + LM;         // bits enumerated by the add-min block
constexpr int LW_MAX = 10;               // walk bits per thread (runtime Lw <= LW_MAX)
constexpr int MIN_CHUNK_BITS = LOWBITS + 5;   // one warp, no walk: 2^15 configurations
constexpr int N_DIRECT_MAX = MIN_CHUNK_BITS - 1;   // N <= 14: direct kernel
constexpr int WQ_BITS = 27;              // sum|Jq| + sum|hq| <= 2^27 grid units
constexpr int TAU_INF = 0x3fffffff;      // "no threshold yet"; every grid energy is far below it
constexpr unsigned long long Q_MAX = ~0ull;

// Sign convention of the field term (reading G2): +1 implements eq. (1) AS PRINTED, H = -sum J s s - sum h s
// (PAPER.md:43), whose fields-only ground state is s_i = +sign(h_i). The other reading some texts use,
// H' = -sum J s s + sum h s = H(J, -h), is this constant set to -1: it is applied wherever h enters the library --
// the quantised fields hq (stage.cu), the fp64 re-evaluation (select.cu) and the QUBO conversion (stage.cu).
constexpr double FIELD_TERM_SIGN = 1.0;

constexpr unsigned POOL_CAP_LOG2 = 22;
constexpr unsigned POOL_CAP = 1u << POOL_CAP_LOG2;     // entries in each of the two candidate pools (64 MiB each)
constexpr unsigned KEEP_CAP = 1u << 20;                // most entries kept after a selection
constexpr int SORT_TILE = 4096;                        // entries sorted by one block in shared memory
constexpr int SORT_THREADS = 1024;

constexpr int HIST_COARSE = 256;                       // coarse bins: 256 fine bins each
constexpr int HIST_FINE = 65536;                       // fine bins over [-Wq, +Wq]
constexpr int HIST_WORDS = HIST_COARSE + HIST_FINE;    // hist[0..256) coarse, hist[256..) fine
constexpr int MAX_SEGMENTS = 64;
constexpr int WALK_THREADS = 256;                      // threads per block of the enumeration kernels
constexpr int WALK_WARPS = WALK_THREADS / 32;

// One candidate: sortable 64-bit key (grid energy or fp64 energy, order preserving) and the state index.
struct __align__(16) Entry {
    unsigned long long key;
    unsigned long long q;
};

__host__ __device__ inline bool entry_less(const Entry& a, const Entry& b)
{
    return a.key < b.key || (a.key == b.key && a.q < b.q);
}
__host__ __device__ inline unsigned long long key_from_i32(int e)
{
    return (unsigned long long)((unsigned)e ^ 0x80000000u);
}
__host__ __device__ inline int i32_from_key(unsigned long long k)
{
    return (int)((unsigned)k ^ 0x80000000u);
}
__device__ inline unsigned long long key_from_f64(double x)
{
    x += 0.0;                                    // -0.0 -> +0.0
    unsigned long long b = (unsigned long long)__double_as_longlong(x);
    return (b >> 63) ? ~b : (b | 0x8000000000000000ull);
}
__device__ inline double f64_from_key(unsigned long long k)
{
    unsigned long long b = (k >> 63) ? (k & 0x7fffffffffffffffull) : ~k;
    return __longlong_as_double((long long)b);
}

// The filter threshold is ONE 64-bit word so that it can be published with a single atomicMin and read with a single
// load:  tau = key32(tauE) << 32 | Qc.   A configuration (e, q) passes iff  e < tauE  or  (e == tauE and q < tauQ),
// tauQ = q_begin + (Qc << qshift), Qc = 0xffffffff meaning "no limit on q". A SMALLER word is a TIGHTER threshold.
constexpr unsigned QC_NONE = 0xffffffffu;
__host__ __device__ inline unsigned long long tau_pack(int tauE, unsigned qc)
{
    return (key_from_i32(tauE) << 32) | (unsigned long long)qc;
}
__host__ __device__ inline int tau_energy(unsigned long long tau) { return i32_from_key(tau >> 32); }
__host__ __device__ inline unsigned tau_qc(unsigned long long tau) { return (unsigned)tau; }

// Device-resident control block of one call; the host reads it back through pinned memory.
struct Ctrl {
    int status;            // ISING_OK or an ISING_ERR_* found by the staging kernel
    int p;                 // grid exponent: weights are multiples of 2^-p
    int exact;             // 1: every weight is on the grid (epsilon = 0)
    int band;              // guard band in grid units: candidates are kept up to E_S + band
    double epsilon;        // bound on |grid energy * 2^-p - eq.(1) energy|
    double W;              // sum_{i<j}|J_ij| + sum_i|h_i|
    long long Wq;          // sum_{i<j}|Jq_ij| + sum_i|hq_i|: every grid energy lies in [-Wq, +Wq]
    unsigned count;        // entries in the pool (kept prefix + new candidates); pushes beyond POOL_CAP are dropped
    unsigned kept;         // entries of the sorted prefix after the last selection
    unsigned long long tau;        // filter threshold word (tau_pack)
    int shift16;           // copy of Tables::shift16 (written by tables_kernel) for the host's statistics
    int hist_shift;        // histogram bin of grid energy e:  (e + Wq) >> hist_shift   (fine bin, < HIST_FINE)
    unsigned band_overflow;    // selection wanted to keep more than KEEP_CAP entries (sticky)
    unsigned pool_overflow;    // a push did not fit into the pool (sticky): the run is void and is redone piecewise
    unsigned long long next_unit;      // work queue: next unit to hand out
    unsigned long long done_configs;   // configurations of completed units (ramp-up rule, see Segment::need_done)
    unsigned count2;           // entries of the compacted pool
    unsigned final_state;      // written by final_small_kernel: 0 not run, 1 done, 2 too many entries for one block
    int eS;                    // S-th smallest grid energy at the final selection (for the band pass)
    unsigned n_sure;           // band pass: entries below the band (certainly among the S lowest)
    unsigned blocks_done;      // direct kernel: blocks that have finished (the last one derives the threshold)
    unsigned pad0;
    unsigned long long hits;   // 1024-configuration blocks that passed the screen and were formed exactly
    unsigned long long false_hits;     // ... of which none passed the exact test
    unsigned long long z_steps;        // tensor-core screen (zscreen.cu): 2^14-configuration blocks screened
    unsigned long long z_flagged;      // ... of which flagged (formed exactly as 16 blocks of 1024)
};

// Instance tables in grid units, built once per call by build_tables (stage.cu).
struct Tables {
    int Jq[64 * 64];               // quantised couplings, row-major, N x N used with stride 64
    int hq[64];
    int C[NMID * NLO];             // C[mid][lo]  = -4 sum_{i in lo, j in mid} Jq_ij        (eq. (2) pair terms)
    int QL[NLO];                   // QL[lo]      = -4 sum_{i<j in lo} Jq_ij
    int QM[NMID];                  // QM[mid]     = -4 sum_{i<j in mid} Jq_ij
    int DV[LW_MAX * 2 * NLO];      // DV[k][sb][lo]  = sgn * -4 sum_{i in lo} Jq[i][w_k],  sgn = sb ? +1 : -1
    int DU[LW_MAX * 2 * NMID];     // DU[k][sb][mid] = sgn * -4 sum_{j in mid} Jq[j][w_k]
    int DW[1 << LW_MAX];           // DW[t] = -sgn_t * 4 sum_{j in R_t} Jq[w_k][w_j]   (walk-internal part of step t)
    // ---- packed 16-bit screening tables of enumerate16.cu: two configurations per 32-bit word, in units of
    //      2^shift16 grid units, every entry rounded DOWN (floor), so sums of them are lower bounds ----
    int shift16;                   // s: one 16-bit unit = 2^s grid units (0 for small-integer instances: exact)
    int cU16;                      // offset added to every 16-bit U entry so that it is never negative
    int cC16;                      // same for the C entries
    int bV16;                      // same for the V entries (both register sets)
    unsigned Cp[(NMID / 2) * NLO]; // Cp[u][lo]  = pack( (C[m0][lo] >> s) + cC , (C[m0 | 8][lo] >> s) + cC ),  m0 = (u & 7) | ((u >> 3) << 4)
    unsigned DVp[LW_MAX * 2 * NLO];        // DVp[k][sb][lo] = +-(DV[k][1][lo] >> s) * 65537    (both halves alike)
    unsigned DUp[LW_MAX * 2 * (NMID / 2)]; // DUp[k][sb][u]  = +-((DU[k][1][m0] >> s) + 65536 (DU[k][1][m0 | 8] >> s))
};

// Tables of the tensor-core screen (zscreen.cu), built once per call by ztables_kernel.
constexpr int ZB = 14;                 // block bits of the screen: lo = spins 0..6 (K), mid = spins 7..13 (N)
struct ZTables {
    uint4 Tb[2048];                    // bf16 T[mid][lo] = 2^(-lambda C'(lo,mid) + t0) in the UMMA canonical K-major layout
    int DPhi[LW_MAX * 16];             // DPhi[k][i] = 2 Jq[i][ZB + k]: change of Phi_i when walk bit k turns on
    int DWz[1 << LW_MAX];              // walk-internal part of Gray step t for walk spins ZB + k (cf. Tables::DW)
    int Cz[1 << ZB];                   // C'(lo | mid << 7) = -4 sum_{a<b set} Jq_ab, grid units
    float lambda;                      // bits per grid unit
    float t0;                          // centres log2 T in [-THETA, +THETA]
    int cmin, cmax;
};

// One segment of the work plan: n_units units of 2^unit_bits configurations starting at state q0.
struct Segment {
    unsigned long long q0;
    unsigned long long first_unit;     // index of the segment's first unit in the queue
    unsigned long long n_units;
    unsigned long long need_done;      // a unit of this segment starts only after this many configurations are done:
                                       // the threshold is then good enough for most blocks to fail the screen
    int unit_bits;                     // 10: one exactly formed 1024-configuration block; 15 + Lw: a walked unit
    int pad;
};

// The work plan of one launch of the enumeration kernel (a kernel parameter: lives in the constant bank).
struct Plan {
    Segment seg[MAX_SEGMENTS];
    unsigned long long total_units;
    unsigned long long q_begin;        // first state of the CALL (origin of the coarse tie limit Qc)
    unsigned long long q_end;          // one past the last state this launch enumerates
    int nseg;
    int N;
    int S;
    int use_hist;                      // 1: pushes feed the histogram and the kernel refreshes tau itself
    int refresh;                       // refresh tau whenever the pool count crosses a multiple of this
    int qshift;                        // tauQ = q_begin + (Qc << qshift)
    int loE;                           // band pass: only configurations with grid energy >= loE are pushed
    unsigned keep_cap;                 // most entries a selection keeps (KEEP_CAP; smaller only in tests of the band pass)
};

// stage.cu
void launch_stage(const double* J, const double* h, int N, Tables* tab, Ctrl* ctrl, unsigned* hist, cudaStream_t st,
                  double extra_eps_rel);
void launch_qubo_to_ising(const double* a, const double* b, int N, double* J, double* h, cudaStream_t st);
// enumerate.cu / enumerate16.cu: the persistent enumeration kernel, int32 and packed 16-bit variants
void launch_walk32(const Tables* tab, Ctrl* ctrl, Entry* pool, unsigned* hist, const Plan& plan, cudaStream_t st);
void launch_walk16(const Tables* tab, Ctrl* ctrl, Entry* pool, unsigned* hist, const Plan& plan, cudaStream_t st);
void launch_direct(const Tables* tab, Ctrl* ctrl, Entry* pool, unsigned* hist, int N, int S, unsigned count,
                   int use_hist, cudaStream_t st);
// zscreen.cu: the tensor-core (tcgen05) screen
void launch_ztables(const Tables* tab, const Ctrl* ctrl, ZTables* zt, int N, cudaStream_t st);
void launch_zwalk(const Tables* tab, const ZTables* zt, Ctrl* ctrl, Entry* pool, unsigned* hist, const Plan& plan,
                  cudaStream_t st);
void set_zscreen_attributes();
void launch_zselftest(unsigned seed, double* out_dev, cudaStream_t st);
// select.cu
int  launch_select(Entry* pool, Ctrl* ctrl, unsigned n, int S, const Plan& plan, cudaStream_t st);   // returns kernels launched
int  launch_compact(const Entry* pool, Entry* pool2, Ctrl* ctrl, const Plan& plan, cudaStream_t st);
int  launch_final_small(const double* J, const double* h, int N, int mode, Entry* pool2, Ctrl* ctrl, int S,
                        unsigned keep_cap, unsigned long long* states_out, double* energies_out, cudaStream_t st);
int  launch_final(const double* J, const double* h, int N, int mode, Entry* pool, unsigned m, int S,
                  unsigned long long* states_out, double* energies_out, cudaStream_t st);
void launch_energies(const double* J, const double* h, int N, int mode, const unsigned long long* states,
                     long long n, double* out, cudaStream_t st);
int  launch_merge_lists(const unsigned long long* states, const double* energies, long long n, int S, Entry* scratch,
                        unsigned long long* states_out, double* energies_out, cudaStream_t st);
int  launch_expand_complements(const unsigned long long* states, const double* energies, int n, int N, int S,
                               Entry* scratch, unsigned long long* states_out, double* energies_out, cudaStream_t st);
int  launch_alg1_chunk(const double* J, const double* h, int N, unsigned long long base, unsigned count,
                       Entry* pool, unsigned kept, cudaStream_t st);
int  launch_emit(const Entry* pool, int S, unsigned long long* states_out, double* energies_out, cudaStream_t st);
int  launch_band_drain(const double* J, const double* h, int N, int mode, Entry* pool, Ctrl* ctrl, unsigned kept,
                       unsigned n, unsigned want, cudaStream_t st);
void set_select_attributes();
// dos.cu
void launch_dos(const Tables* tab, int N, int Lw, unsigned long long base, unsigned nthreads, int e_lo, int bshift,
                int nbins, unsigned long long* hist, cudaStream_t st);
void launch_dos_direct(const Tables* tab, int N, int e_lo, int bshift, unsigned long long* hist, cudaStream_t st);
// peak.cu
double run_fma_peak(double ms_target, cudaStream_t st, int which);
// api.cu: the calling thread's detail string behind ising_last_error(), for entry points that live in other files
void set_last_error(const char* what);

}  // namespace ising
