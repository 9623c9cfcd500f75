/*
 * oracle_gray.c -- TEST INFRASTRUCTURE, NOT THE PRODUCT.  Tier-2 oracle for INTEGER-weight instances only.
 *
 * Same result as oracle.c (the S lowest (E, q) pairs of eq. (1), ascending under (E, q)), reached by
 * the textbook single-spin-flip recurrence instead of the O(N^2) sum per state, so that BASELINE.json config 4
 * (N = 40, 2^40 states, 107 edges) finishes in minutes on a few cores. It exists only to write the stored expected
 * output tests/golden/cfg4.txt; SURVEY.md section 8(c) lists it as pin P14 ("optional tier-2 oracle").
 *
 * It is NOT the definition: oracle.c is. It is trusted only as far as tests/test_oracle_pins.py pins it to oracle.c
 * (identical lists on random integer instances N <= 22 of several densities, on heavy-tie instances, on range
 * splits, and on config 2's stored golden, which oracle.c wrote). It shares no code with oracle.c beyond the
 * conventions below, and none with paper_1904_03621_b200/csrc (the CUDA path).
 *
 * Algorithm (every quantity an exact int64; integer inputs are required and checked):
 *   slab of 2^k consecutive states, k <= N, base = first state (low k bits zero); visit q = base | gray(t),
 *   gray(t) = t ^ (t >> 1), t = 0 .. 2^k - 1: consecutive t differ in the single spin f = ctz(t).
 *   E(q) and the local fields  phi_i = h_i + sum_j J_ij s_j  are computed directly (eq. (1)) at t = 0; flipping
 *   spin f:   E += 2 s_f phi_f   (the terms of eq. (1) that contain s_f are  -s_f phi_f),   s_f = -s_f,
 *             phi_j += 2 J_jf s_f(new)   for every neighbour j of f.
 *   Every visited (E, q) is offered to a size-S max-heap under the total order (E, q) (reading G4).
 * Conventions: bit i of q <-> spin i, 0 <-> s = -1 (G1); both terms of eq. (1) carry a minus
 * sign (G2); each unordered pair once, coupling J[i*N+j].
 */
#include <stdint.h>
#include <stdlib.h>
#include <string.h>
#include <math.h>
#ifdef _OPENMP
#include <omp.h>
#endif

typedef struct { int64_t e; uint64_t q; } gpair_t;

static int gless(gpair_t a, gpair_t b) { return a.e < b.e || (a.e == b.e && a.q < b.q); }
static int gcmp(const void *pa, const void *pb)
{
    gpair_t a = *(const gpair_t *)pa, b = *(const gpair_t *)pb;
    return gless(a, b) ? -1 : (gless(b, a) ? 1 : 0);
}

typedef struct { gpair_t *a; int64_t n, cap; } gheap_t;

static void gheap_offer(gheap_t *H, gpair_t p)
{
    if (H->n < H->cap) {
        int64_t i = H->n++;
        H->a[i] = p;
        while (i > 0) {
            int64_t par = (i - 1) / 2;
            if (!gless(H->a[par], H->a[i])) break;
            gpair_t t = H->a[i]; H->a[i] = H->a[par]; H->a[par] = t;
            i = par;
        }
    } else if (gless(p, H->a[0])) {
        int64_t i = 0;
        H->a[0] = p;
        for (;;) {
            int64_t l = 2 * i + 1, r = l + 1, m = i;
            if (l < H->n && gless(H->a[m], H->a[l])) m = l;
            if (r < H->n && gless(H->a[m], H->a[r])) m = r;
            if (m == i) break;
            gpair_t t = H->a[i]; H->a[i] = H->a[m]; H->a[m] = t;
            i = m;
        }
    }
}

/*
 * The S lowest (E, q) of q_begin <= q < q_end for an integer-weight instance. q_begin and q_end must be multiples
 * of 2^slab_bits (slab_bits <= N). Returns the number of pairs written (min(S, q_end - q_begin)), -1 on bad
 * arguments, -2 if some weight is not an integer or sum|J| + sum|h| >= 2^52.
 */
int64_t oracle_gray_lowest(const double *J, const double *h, int N, int64_t S, uint64_t q_begin, uint64_t q_end,
                           int slab_bits, uint64_t *states_out, double *energies_out, int threads)
{
    if (!J || !h || !states_out || !energies_out) return -1;
    if (N < 1 || N > 63 || S < 1 || q_end < q_begin || q_end > (1ull << N)) return -1;
    if (slab_bits < 0 || slab_bits > N) return -1;
    const uint64_t slab = 1ull << slab_bits;
    if ((q_begin % slab) || (q_end % slab)) return -1;
    if (q_end == q_begin) return 0;

    /* integer check and integer copies */
    int64_t *Ji = (int64_t *)malloc(sizeof(int64_t) * (size_t)N * (size_t)N);
    int64_t hi[64];
    int nbr[64][64], deg[64];
    if (!Ji) return -1;
    double W = 0.0;
    for (int i = 0; i < N; ++i) {
        if (h[i] != floor(h[i]) || !isfinite(h[i])) { free(Ji); return -2; }
        hi[i] = (int64_t)h[i];
        W += fabs(h[i]);
        deg[i] = 0;
        for (int j = 0; j < N; ++j) {
            double v = J[(size_t)i * N + j];
            if (v != floor(v) || !isfinite(v)) { free(Ji); return -2; }
            Ji[(size_t)i * N + j] = (int64_t)v;
            if (i < j) W += fabs(v);
            if (i != j && v != 0.0) nbr[i][deg[i]++] = j;
        }
    }
    if (W >= 4503599627370496.0) { free(Ji); return -2; }

    const uint64_t nslabs = (q_end - q_begin) >> slab_bits;
    int nt = 1;
#ifdef _OPENMP
    nt = threads > 0 ? threads : omp_get_max_threads();
#endif
    if ((uint64_t)nt > nslabs) nt = (int)nslabs;
    gpair_t *all = (gpair_t *)malloc(sizeof(gpair_t) * (size_t)nt * (size_t)S);
    int64_t *cnt = (int64_t *)calloc((size_t)nt, sizeof(int64_t));
    if (!all || !cnt) { free(Ji); free(all); free(cnt); return -1; }

#pragma omp parallel num_threads(nt)
    {
        int tid = 0;
#ifdef _OPENMP
        tid = omp_get_thread_num();
#endif
        gheap_t H; H.a = all + (size_t)tid * (size_t)S; H.n = 0; H.cap = S;
        int64_t s[64], phi[64];
#pragma omp for schedule(dynamic, 1)
        for (int64_t sl = 0; sl < (int64_t)nslabs; ++sl) {
            const uint64_t base = q_begin + ((uint64_t)sl << slab_bits);
            /* t = 0: eq. (1) and the local fields directly */
            for (int i = 0; i < N; ++i) s[i] = ((base >> i) & 1ull) ? 1 : -1;
            int64_t E = 0;
            for (int i = 0; i < N; ++i) {
                for (int j = i + 1; j < N; ++j) E -= Ji[(size_t)i * N + j] * s[i] * s[j];
                E -= hi[i] * s[i];
                int64_t f = hi[i];
                for (int j = 0; j < N; ++j) f += Ji[(size_t)i * N + j] * s[j];     /* J_ii = 0 */
                phi[i] = f;
            }
            gpair_t p; p.e = E; p.q = base;
            gheap_offer(&H, p);
            for (uint64_t t = 1; t < slab; ++t) {
                const int f = __builtin_ctzll(t);
                E += 2 * s[f] * phi[f];
                s[f] = -s[f];
                const int64_t two_s = 2 * s[f];
                for (int a = 0; a < deg[f]; ++a) {
                    const int j = nbr[f][a];
                    phi[j] += Ji[(size_t)j * N + f] * two_s;
                }
                p.e = E; p.q = base | (t ^ (t >> 1));
                if (H.n < H.cap || gless(p, H.a[0])) gheap_offer(&H, p);
            }
        }
        cnt[tid] = H.n;
    }
    size_t m = 0;
    for (int t = 0; t < nt; ++t) {
        memmove(all + m, all + (size_t)t * (size_t)S, sizeof(gpair_t) * (size_t)cnt[t]);
        m += (size_t)cnt[t];
    }
    qsort(all, m, sizeof(gpair_t), gcmp);
    int64_t n_out = (int64_t)(m < (size_t)S ? m : (size_t)S);
    for (int64_t r = 0; r < n_out; ++r) { states_out[r] = all[r].q; energies_out[r] = (double)all[r].e; }
    free(Ji); free(all); free(cnt);
    return n_out;
}
