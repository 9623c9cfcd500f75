/*
 * oracle_bnb.c -- TEST INFRASTRUCTURE, NOT THE PRODUCT.  Tier-3 oracle: exact branch and bound.
 *
 * Same result as oracle.c -- the S lowest (E, q) pairs of eq. (1), ascending under (E, q) -- reached
 * WITHOUT visiting all 2^N states, so that BASELINE.json config 5 (N = 48, 2^48 states; about 150 days for
 * oracle.c) gets a complete stored list, tests/golden/cfg5.txt. A depth-first search fixes the spins one at a time
 * and discards a subtree only when a rigorous lower bound on every energy in it exceeds the K-th best energy found
 * so far: nothing that could belong to the answer is ever discarded, so the result is exact, not heuristic.
 *
 * It is NOT the definition: oracle.c is. It is trusted only as far as tests/test_oracle_pins.py pins it to oracle.c:
 * identical lists on random real and integer instances up to N = 24, on heavy-tie instances, and on the stored lists
 * of configs 1 and 3 (N = 36), which oracle.c wrote. It shares no code with oracle.c beyond the conventions, and
 * none with paper_1904_03621_b200/csrc (the CUDA path); no input of it comes from the CUDA path.
 *
 * Search.  Spins are fixed in the order ord[0], ord[1], ... (decreasing |h_i| + sum_j |J_ij|). With the set F fixed:
 *     E_F     = - sum_{i<j in F} J_ij s_i s_j - sum_{i in F} h_i s_i          (the part of eq. (1) inside F)
 *     phi_i   = h_i + sum_{j in F} J_ij s_j                                   (field of F on a free spin i)
 *     E(s)    = E_F - sum_{i free} s_i phi_i - sum_{i<j free} J_ij s_i s_j
 *            >= E_F - sum_{i free} |phi_i| - sum_{i<j free} |J_ij|  =: LB      (every term at its most negative)
 * A subtree is cut iff LB > tau + margin, tau = the K-th best energy found so far (K = S + spare), margin =
 * 1e-9 (W + 1) >> the fp64 rounding of the incrementally accumulated E_F and LB (about 1e-13 W). The more
 * promising value s = sign(phi) is tried first, so good states are found early and tau tightens quickly.
 * The K kept states are then re-evaluated by eq. (1) in oracle.c's summation order (pairs i<j row-major, then
 * fields) and sorted under (E, q): the energies written out are bit-identical to oracle.c's.
 * Exactness of the K boundary: states whose energies differ by less than `margin` could swap across rank K; the
 * caller asks for spare entries beyond S for that reason (and config 5's lowest levels are >= 1e-5 apart).
 *
 * Parallelism: the first `split` levels are expanded into 2^split subtrees handed to OpenMP threads; each thread
 * keeps its own K-heap; tau is shared (any thread's K-th best is an upper bound on the global K-th best).
 */
#include <stdint.h>
#include <stdlib.h>
#include <string.h>
#include <math.h>
#ifdef _OPENMP
#include <omp.h>
#endif

typedef struct { double e; uint64_t q; } bpair_t;

static int bless(bpair_t a, bpair_t b) { return a.e < b.e || (a.e == b.e && a.q < b.q); }
static int bnb_cmp(const void *pa, const void *pb)
{
    bpair_t a = *(const bpair_t *)pa, b = *(const bpair_t *)pb;
    return bless(a, b) ? -1 : (bless(b, a) ? 1 : 0);
}

typedef struct { bpair_t *a; int64_t n, cap; } bheap_t;

static void bheap_offer(bheap_t *H, bpair_t p)
{
    if (H->n < H->cap) {
        int64_t i = H->n++;
        H->a[i] = p;
        while (i > 0) {
            int64_t par = (i - 1) / 2;
            if (!bless(H->a[par], H->a[i])) break;
            bpair_t t = H->a[i]; H->a[i] = H->a[par]; H->a[par] = t;
            i = par;
        }
    } else if (bless(p, H->a[0])) {
        int64_t i = 0;
        H->a[0] = p;
        for (;;) {
            int64_t l = 2 * i + 1, r = l + 1, m = i;
            if (l < H->n && bless(H->a[m], H->a[l])) m = l;
            if (r < H->n && bless(H->a[m], H->a[r])) m = r;
            if (m == i) break;
            bpair_t t = H->a[i]; H->a[i] = H->a[m]; H->a[m] = t;
            i = m;
        }
    }
}

typedef struct {
    int N;
    const double *Jo;          /* couplings permuted into search order: Jo[a*N+b] = J[ord[a]][ord[b]] */
    const double *ho;          /* fields in search order */
    const int *ord;            /* search position -> original spin index */
    const double *pairs_below; /* pairs_below[d] = sum_{d <= a < b < N} |Jo[a][b]| */
    double margin;
    volatile double *tau;      /* shared K-th best energy (upper bound) */
    uint64_t nodes;
} bctx_t;

/* depth-first search below depth d; phi = fields of the fixed set on spins d..N-1 (search order), E = E_F */
static void bnb_dfs(bctx_t *C, bheap_t *H, int d, double E, const double *phi, uint64_t q, double *work)
{
    const int N = C->N;
    const double *Jo = C->Jo;
    double *next = work + (size_t)d * N;               /* this level's scratch: fields after fixing spin d */
    const int first = phi[d] >= 0.0 ? 1 : -1;          /* s = sign(phi) lowers the energy: try it first */
    for (int t = 0; t < 2; ++t) {
        const int s = t == 0 ? first : -first;
        const double E1 = E - s * phi[d];
        double lb = E1 - C->pairs_below[d + 1];
        for (int i = d + 1; i < N; ++i) {
            const double f = phi[i] + Jo[(size_t)i * N + d] * s;
            next[i] = f;
            lb -= fabs(f);
        }
        ++C->nodes;
        if (lb > *C->tau + C->margin) continue;         /* nothing below can be among the K lowest */
        const uint64_t q1 = s > 0 ? (q | (1ull << C->ord[d])) : q;
        if (d + 1 == N) {
            bpair_t p; p.e = E1; p.q = q1;
            bheap_offer(H, p);
            if (H->n == H->cap && H->a[0].e < *C->tau) {
#pragma omp critical(bnb_tau)
                { if (H->a[0].e < *C->tau) *C->tau = H->a[0].e; }
            }
        } else {
            bnb_dfs(C, H, d + 1, E1, next, q1, work);
        }
    }
}

/*
 * The S lowest (E, q) of the whole space by exact branch and bound. Internally K = S + spare states are kept.
 * Writes min(K, 2^N) pairs (ascending under (E, q), energies by eq. (1) in oracle.c's summation order) and returns
 * that count; -1 on bad arguments. nodes_out (optional) receives the number of search nodes visited.
 */
int64_t oracle_bnb_lowest(const double *J, const double *h, int N, int64_t S, int64_t spare,
                          uint64_t *states_out, double *energies_out, int threads, uint64_t *nodes_out)
{
    if (!J || !h || !states_out || !energies_out) return -1;
    if (N < 1 || N > 63 || S < 1 || spare < 0) return -1;
    int64_t K = S + spare;
    if (N < 62 && K > ((int64_t)1 << N)) K = (int64_t)1 << N;

    /* search order: decreasing |h_i| + sum_j |J_ij| */
    int ord[64];
    double weight[64], W = 0.0;
    for (int i = 0; i < N; ++i) {
        double w = fabs(h[i]);
        for (int j = 0; j < N; ++j) if (j != i) w += fabs(J[(size_t)i * N + j]);
        weight[i] = w;
        ord[i] = i;
        W += fabs(h[i]);
        for (int j = i + 1; j < N; ++j) W += fabs(J[(size_t)i * N + j]);
    }
    for (int a = 1; a < N; ++a) {                        /* insertion sort, stable */
        int x = ord[a], b = a;
        while (b > 0 && weight[ord[b - 1]] < weight[x]) { ord[b] = ord[b - 1]; --b; }
        ord[b] = x;
    }
    double *Jo = (double *)malloc(sizeof(double) * (size_t)N * (size_t)N);
    double ho[64], pairs_below[65];
    if (!Jo) return -1;
    for (int a = 0; a < N; ++a) {
        ho[a] = h[ord[a]];
        for (int b = 0; b < N; ++b) Jo[(size_t)a * N + b] = a == b ? 0.0 : J[(size_t)ord[a] * N + ord[b]];
    }
    pairs_below[N] = 0.0;
    for (int d = N - 1; d >= 0; --d) {
        double acc = pairs_below[d + 1];
        for (int b = d + 1; b < N; ++b) acc += fabs(Jo[(size_t)d * N + b]);
        pairs_below[d] = acc;
    }

    int nt = 1;
#ifdef _OPENMP
    nt = threads > 0 ? threads : omp_get_max_threads();
#endif
    int split = N > 16 ? 12 : (N > 4 ? N - 4 : 0);      /* 2^split subtrees */
    const int64_t nsub = (int64_t)1 << split;
    if (nt > nsub) nt = (int)nsub;
    bpair_t *all = (bpair_t *)malloc(sizeof(bpair_t) * (size_t)nt * (size_t)K);
    int64_t *cnt = (int64_t *)calloc((size_t)nt, sizeof(int64_t));
    if (!all || !cnt) { free(Jo); free(all); free(cnt); return -1; }
    volatile double tau = INFINITY;
    uint64_t nodes_total = 0;

#pragma omp parallel num_threads(nt) reduction(+ : nodes_total)
    {
        int tid = 0;
#ifdef _OPENMP
        tid = omp_get_thread_num();
#endif
        bheap_t H; H.a = all + (size_t)tid * (size_t)K; H.n = 0; H.cap = K;
        bctx_t C;
        C.N = N; C.Jo = Jo; C.ho = ho; C.ord = ord; C.pairs_below = pairs_below;
        C.margin = 1e-9 * (W + 1.0); C.tau = &tau; C.nodes = 0;
        double *work = (double *)malloc(sizeof(double) * (size_t)(N + 1) * (size_t)N);
        double *phi0 = (double *)malloc(sizeof(double) * (size_t)N);
#pragma omp for schedule(dynamic, 1)
        for (int64_t sub = 0; sub < nsub; ++sub) {
            /* walk the prefix: spin d takes the value given by bit d of sub, with the same bound test */
            for (int i = 0; i < N; ++i) phi0[i] = ho[i];
            double E = 0.0;
            uint64_t q = 0;
            int alive = 1;
            for (int d = 0; d < split && alive; ++d) {
                const int s = (sub >> d) & 1 ? 1 : -1;
                E -= s * phi0[d];
                double lb = E - pairs_below[d + 1];
                for (int i = d + 1; i < N; ++i) { phi0[i] += Jo[(size_t)i * N + d] * s; lb -= fabs(phi0[i]); }
                if (s > 0) q |= 1ull << ord[d];
                ++C.nodes;
                if (lb > tau + C.margin) alive = 0;
            }
            if (!alive) continue;
            if (split == N) {
                bpair_t p; p.e = E; p.q = q;
                bheap_offer(&H, p);
            } else {
                bnb_dfs(&C, &H, split, E, phi0, q, work);
            }
        }
        cnt[tid] = H.n;
        nodes_total += C.nodes;
        free(work); free(phi0);
    }

    /* gather, re-evaluate by eq. (1) in the canonical order (pairs i<j row-major, then fields), sort, emit K */
    size_t m = 0;
    for (int t = 0; t < nt; ++t) {
        memmove(all + m, all + (size_t)t * (size_t)K, sizeof(bpair_t) * (size_t)cnt[t]);
        m += (size_t)cnt[t];
    }
    for (size_t r = 0; r < m; ++r) {
        double s[64], acc = 0.0;
        for (int i = 0; i < N; ++i) s[i] = ((all[r].q >> i) & 1ull) ? 1.0 : -1.0;
        for (int i = 0; i < N; ++i)
            for (int j = i + 1; j < N; ++j) acc += -(s[i] * s[j]) * J[(size_t)i * N + j];
        for (int i = 0; i < N; ++i) acc += -s[i] * h[i];
        all[r].e = acc;
    }
    qsort(all, m, sizeof(bpair_t), bnb_cmp);
    int64_t n_out = (int64_t)(m < (size_t)K ? m : (size_t)K);
    for (int64_t r = 0; r < n_out; ++r) { states_out[r] = all[r].q; energies_out[r] = all[r].e; }
    if (nodes_out) *nodes_out = nodes_total;
    free(Jo); free(all); free(cnt);
    return n_out;
}
