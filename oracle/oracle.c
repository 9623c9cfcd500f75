/*
 * oracle.c -- TEST INFRASTRUCTURE, NOT THE PRODUCT.
 *
 * Plain, slow, obviously-correct CPU definition of what the hot path of
 * arXiv 1904.03621 computes: over every spin configuration q of an Ising model,
 * the energy of eq. (1), and the S lowest (energy, q) pairs in
 * ascending order (PAPER.md:9 abstract, "sort_by_key").
 *
 * Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference
 * legs may build, load or call this file. It shares no code, header, table or helper
 * with paper_1904_03621_b200/csrc (the CUDA path) and includes nothing from it.
 *
 * Readings of the paper used here:
 *   G1  bit i (LSB = bit 0) of q  <->  spin s_i,  bit 0 <-> s_i = -1, bit 1 <-> s_i = +1
 *       (q = (s+1)/2; "s_i = -1 [or q_i = 0]").
 *   G2  both terms of eq. (1) carry a minus sign, literally as printed.
 *   G4  ties: total order (E, q) ascending.
 *   <i,j> runs over each unordered pair once: i < j, coupling J[i*N+j].
 *
 * Arithmetic: IEEE fp64, fixed summation order (pairs in row-major i<j order, then fields).
 * Multiplying by s_i*s_j = +-1 is exact, so FMA contraction cannot change a result.
 * For integer-valued J, h every partial sum is an exactly representable integer.
 *
 * Pins (tests/test_oracle_pins.py, all run with -m "not gpu"):
 *   oracle_energy  : Listing-1 instance by hand (tests/golden/listing1.txt), ferromagnet and
 *                    Mattis closed forms, fields-only, chain, QUBO identity eqs. (2),(3), h=0 symmetry.
 *   oracle_lowest  : the same closed-form spectra incl. tie order, full sort for N <= 16,
 *                    decoupled-blocks pair-sum construction, range splitting.
 *   oracle_dos     : binomial level counts (uniform field, uniform ferromagnet).
 * Faster exact oracles for the configs this one cannot finish live in oracle_gray.c and oracle_bnb.c; both are
 * pinned to this file and neither replaces it as the definition.
 */
#include <stdint.h>
#include <stdlib.h>
#include <string.h>
#include <math.h>
#ifdef _OPENMP
#include <omp.h>
#endif

/* G2: sign in front of the field term of eq. (1). -1.0 = as printed in the paper. */
#define ORACLE_FIELD_SIGN (-1.0)
/* sign in front of the coupling term of eq. (1). */
#define ORACLE_COUPLING_SIGN (-1.0)

/* eq. (1):  H(s) = - sum_{i<j} J_ij s_i s_j - sum_i h_i s_i */
double oracle_energy(const double *J, const double *h, int N, uint64_t q)
{
    double s[64];
    for (int i = 0; i < N; ++i)
        s[i] = ((q >> i) & 1ull) ? 1.0 : -1.0;          /* G1 */
    double acc = 0.0;
    for (int i = 0; i < N; ++i)
        for (int j = i + 1; j < N; ++j)
            acc += ORACLE_COUPLING_SIGN * (s[i] * s[j]) * J[(size_t)i * N + j];
    for (int i = 0; i < N; ++i)
        acc += ORACLE_FIELD_SIGN * s[i] * h[i];
    return acc;
}

/* energies of a contiguous run of states (for tests: full sorts, sampled checks) */
void oracle_energies(const double *J, const double *h, int N,
                     uint64_t q_begin, uint64_t count, double *out)
{
#pragma omp parallel for schedule(static)
    for (int64_t t = 0; t < (int64_t)count; ++t)
        out[t] = oracle_energy(J, h, N, q_begin + (uint64_t)t);
}

/* energies of an arbitrary list of states */
void oracle_energies_of(const double *J, const double *h, int N,
                        const uint64_t *q, uint64_t count, double *out)
{
    for (uint64_t t = 0; t < count; ++t)
        out[t] = oracle_energy(J, h, N, q[t]);
}

typedef struct { double e; uint64_t q; } pair_t;

/* total order (E, q), G4 */
static int pair_less(pair_t a, pair_t b)
{
    if (a.e < b.e) return 1;
    if (a.e > b.e) return 0;
    return a.q < b.q;
}
static int pair_cmp(const void *pa, const void *pb)
{
    pair_t a = *(const pair_t *)pa, b = *(const pair_t *)pb;
    if (pair_less(a, b)) return -1;
    if (pair_less(b, a)) return 1;
    return 0;
}

/* size-S max-heap keyed by (E, q): root = the worst pair kept so far */
typedef struct { pair_t *a; int n, cap; } heap_t;

static void heap_sift_down(heap_t *H, int i)
{
    for (;;) {
        int l = 2 * i + 1, r = l + 1, m = i;
        if (l < H->n && pair_less(H->a[m], H->a[l])) m = l;
        if (r < H->n && pair_less(H->a[m], H->a[r])) m = r;
        if (m == i) return;
        pair_t t = H->a[i]; H->a[i] = H->a[m]; H->a[m] = t;
        i = m;
    }
}
static void heap_offer(heap_t *H, pair_t p)
{
    if (H->n < H->cap) {
        int i = H->n++;
        H->a[i] = p;
        while (i > 0) {
            int par = (i - 1) / 2;
            if (!pair_less(H->a[par], H->a[i])) break;
            pair_t t = H->a[i]; H->a[i] = H->a[par]; H->a[par] = t;
            i = par;
        }
    } else if (pair_less(p, H->a[0])) {
        H->a[0] = p;
        heap_sift_down(H, 0);
    }
}

/*
 * The S lowest (E, q) of q_begin <= q < q_end, ascending under (E, q).
 * Writes min(S, q_end - q_begin) pairs; returns that count, or -1 on bad arguments.
 * threads <= 0: all available.
 */
int64_t oracle_lowest(const double *J, const double *h, int N, int64_t S,
                      uint64_t q_begin, uint64_t q_end,
                      uint64_t *states_out, double *energies_out, int threads)
{
    if (!J || !h || !states_out || !energies_out) return -1;
    if (N < 1 || N > 63 || S < 1 || q_end < q_begin) return -1;
    if (q_end > (1ull << N)) return -1;
    uint64_t total = q_end - q_begin;
    if (total == 0) return 0;
    int nt = 1;
#ifdef _OPENMP
    nt = threads > 0 ? threads : omp_get_max_threads();
#endif
    if ((uint64_t)nt > total) nt = (int)total;
    pair_t *all = (pair_t *)malloc(sizeof(pair_t) * (size_t)nt * (size_t)S);
    int *cnt = (int *)calloc((size_t)nt, sizeof(int));
    if (!all || !cnt) { free(all); free(cnt); return -1; }

#pragma omp parallel num_threads(nt)
    {
        int tid = 0;
#ifdef _OPENMP
        tid = omp_get_thread_num();
#endif
        /* contiguous slab of states for this thread */
        uint64_t lo = q_begin + (total / (uint64_t)nt) * (uint64_t)tid
                    + ((uint64_t)tid < total % (uint64_t)nt ? (uint64_t)tid : total % (uint64_t)nt);
        uint64_t len = total / (uint64_t)nt + ((uint64_t)tid < total % (uint64_t)nt ? 1 : 0);
        heap_t H; H.a = all + (size_t)tid * (size_t)S; H.n = 0; H.cap = (int)S;
        for (uint64_t q = lo; q < lo + len; ++q) {
            pair_t p; p.q = q; p.e = oracle_energy(J, h, N, q);
            heap_offer(&H, p);
        }
        cnt[tid] = H.n;
    }
    /* merge: gather all kept pairs, sort ascending, emit the first S */
    size_t m = 0;
    for (int t = 0; t < nt; ++t) {
        memmove(all + m, all + (size_t)t * (size_t)S, sizeof(pair_t) * (size_t)cnt[t]);
        m += (size_t)cnt[t];
    }
    qsort(all, m, sizeof(pair_t), pair_cmp);
    int64_t n_out = (int64_t)(m < (size_t)S ? m : (size_t)S);
    for (int64_t r = 0; r < n_out; ++r) { states_out[r] = all[r].q; energies_out[r] = all[r].e; }
    free(all); free(cnt);
    return n_out;
}

/*
 * Density of states (cf. the paper's Fig. 6): hist[b] = number of states q in [0, 2^N) with
 * e_lo + b*width <= E(q) < e_lo + (b+1)*width, E by eq. (1) as above. Returns the number of states that fell
 * outside [e_lo, e_lo + nbins*width) (they are not counted), or -1 on bad arguments.
 * Pins (tests/test_oracle_pins.py): binomial level counts of the uniform ferromagnet and of a uniform field.
 */
int64_t oracle_dos(const double *J, const double *h, int N, double e_lo, double width, int nbins, uint64_t *hist)
{
    if (!J || !h || !hist || N < 1 || N > 40 || nbins < 1 || !(width > 0.0)) return -1;
    for (int b = 0; b < nbins; ++b) hist[b] = 0;
    const int64_t total = (int64_t)1 << N;
    int64_t outside = 0;
#pragma omp parallel
    {
        uint64_t *loc = (uint64_t *)calloc((size_t)nbins, sizeof(uint64_t));
        int64_t out_loc = 0;
#pragma omp for schedule(static)
        for (int64_t q = 0; q < total; ++q) {
            const double b = floor((oracle_energy(J, h, N, (uint64_t)q) - e_lo) / width);
            if (b < 0.0 || b >= (double)nbins) ++out_loc;
            else ++loc[(int)b];
        }
#pragma omp critical
        {
            for (int b = 0; b < nbins; ++b) hist[b] += loc[b];
            outside += out_loc;
        }
        free(loc);
    }
    return outside;
}

int oracle_max_threads(void)
{
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}
