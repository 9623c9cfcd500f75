// stage.cu -- SURVEY.md section 8 row a1: validate the instance, put it on a power-of-two grid, build the tables.
//
// The enumeration works in exact integer arithmetic on the quantised instance (Jq, hq) = rint((J, h) * 2^p):
// every sum the kernels form is an int32 multiple of 2^-p, so there is no accumulation error and the only
// difference to eq. (1) is the input rounding, bounded rigorously by
//      epsilon = sum_{i<j} |Jq_ij 2^-p - J_ij| + sum_i |hq_i 2^-p - h_i|.
// Integer / dyadic instances have epsilon = 0 and are enumerated exactly.
//
// Tables are the paper's QUBO form, eqs. (2),(3), taken relative to a base state q0 whose
// L, M and W bits are 0:   E(q0 + A) = E(q0) - 2 sum_{i in A} Phi_i(q0) - 4 sum_{i<j in A} J_ij
// with Phi_i(q0) = h_i + sum_j J_ij s_j(q0) the local field at the base state (a_ij = 4 J_ij of eq. (3)).
#include "common.cuh"
#include "../../include/ising.h"

namespace ising {

constexpr int STAGE_THREADS = 1024;

__device__ void build_tables(Tables* __restrict__ tab, Ctrl* __restrict__ ctrl, int N);

__global__ void __launch_bounds__(STAGE_THREADS) stage_kernel(const double* __restrict__ J, const double* __restrict__ h, int N,
                                                    Tables* __restrict__ tab, Ctrl* __restrict__ ctrl,
                                                    unsigned* __restrict__ hist, double extra_eps_rel)
{
    // the candidate histogram of the call starts empty (walk.cuh)
    if (hist)
        for (int i = threadIdx.x; i < HIST_WORDS / 4; i += blockDim.x) reinterpret_cast<uint4*>(hist)[i] = make_uint4(0u, 0u, 0u, 0u);
    __shared__ int s_status;
    __shared__ int s_p;
    __shared__ double s_red[STAGE_THREADS];
    const int tid = threadIdx.x;
    constexpr int NO_ERROR_YET = -1000;
    if (tid == 0) s_status = NO_ERROR_YET;
    __syncthreads();

    // ---- validation: finite, symmetric, zero diagonal (include/ising.h error codes; most severe wins) ----
    int bad = ISING_OK;
    for (int idx = tid; idx < N * N; idx += blockDim.x) {
        int i = idx / N, j = idx % N;
        double v = J[idx];
        if (!isfinite(v)) bad = ISING_ERR_NONFINITE;
        else if (i == j) { if (v != 0.0 && bad != ISING_ERR_NONFINITE) bad = ISING_ERR_DIAGONAL; }
        else if (!(v == J[j * N + i]) && bad == ISING_OK) bad = ISING_ERR_ASYMMETRIC;
    }
    for (int i = tid; i < N; i += blockDim.x)
        if (!isfinite(h[i])) bad = ISING_ERR_NONFINITE;
    // codes are negative; NONFINITE (-4) outranks ASYMMETRIC (-5) outranks DIAGONAL (-6): report the max
    if (bad != ISING_OK) atomicMax(&s_status, bad);
    __syncthreads();
    if (s_status != NO_ERROR_YET) {
        if (tid == 0) ctrl->status = s_status;
        return;
    }

    // ---- W = sum_{i<j}|J_ij| + sum_i|h_i| : per-thread partials, then a fixed-order tree (deterministic) ----
    double part = 0.0;
    for (int idx = tid; idx < N * N; idx += blockDim.x) {
        int i = idx / N, j = idx % N;
        if (i < j) part += fabs(J[idx]);
    }
    for (int i = tid; i < N; i += blockDim.x) part += fabs(h[i]);
    s_red[tid] = part;
    __syncthreads();
    for (int s = STAGE_THREADS / 2; s > 0; s >>= 1) {
        if (tid < s) s_red[tid] += s_red[tid + s];
        __syncthreads();
    }
    const double W = s_red[0];
    // smallest exponent p_req with every weight an integer multiple of 2^-p_req (the instance's own grid):
    // x = M 2^(e-53), M a 53-bit integer  =>  lowest set bit of x has exponent e - 53 + ctz(M)
    __shared__ int s_preq;
    if (tid == 0) s_preq = -100000;
    __syncthreads();
    {
        int req = -100000;
        for (int idx = tid; idx < N * N + N; idx += blockDim.x) {
            const double v = idx < N * N ? J[idx] : h[idx - N * N];
            if (v != 0.0 && isfinite(v)) {
                // |v| = M 2^base with the integer M read straight from the bit pattern (normal: implicit leading one)
                const unsigned long long bits = (unsigned long long)__double_as_longlong(fabs(v));
                const int eb = (int)(bits >> 52);
                const unsigned long long M = (bits & 0xfffffffffffffull) | (eb ? 0x10000000000000ull : 0ull);
                const int low = (eb ? eb - 1075 : -1074) + (__ffsll((long long)M) - 1);
                if (-low > req) req = -low;
            }
        }
        if (req > -100000) atomicMax(&s_preq, req);
    }
    __syncthreads();
    if (tid == 0) {
        int p = 0, st = ISING_OK;
        if (!isfinite(W)) st = ISING_ERR_RANGE_W;
        else if (W > 0.0) {
            int e;
            frexp(W * (1.0 + 1e-9), &e);          // W < 2^e  (the factor covers the rounding of the fp64 sum)
            p = WQ_BITS - e;                      // sum of |rint(x 2^p)| <= W 2^p + (#terms)/2 < 2^27 + 2^11
            if (p > 1000 || p < -1000) st = ISING_ERR_RANGE_W;
            // integer / dyadic instance whose own grid fits: use it (smaller integers, exact and a finer 16-bit screen)
            else if (s_preq <= p && s_preq >= -1000) p = s_preq;
        }
        s_p = p;
        s_status = st;
    }
    __syncthreads();
    if (s_status != ISING_OK) { if (tid == 0) ctrl->status = s_status; return; }
    const int p = s_p;

    // ---- quantise; accumulate the rounding error of each weight that enters eq. (1) once, and the exact integer
    //      sum Wq of the |grid weights| (every grid energy lies in [-Wq, +Wq]) ----
    __shared__ unsigned long long s_wq;
    if (tid == 0) s_wq = 0ull;
    __syncthreads();
    unsigned long long wq = 0ull;
    double err = 0.0;
    // x 2^p and x 2^-p as exact multiplications (|p| <= 1000: both powers are normal doubles)
    const double scale = __longlong_as_double((long long)(p + 1023) << 52);
    const double inv_scale = __longlong_as_double((long long)(1023 - p) << 52);
    for (int idx = tid; idx < 64 * 64; idx += blockDim.x) {
        int i = idx >> 6, j = idx & 63;
        int q = 0;
        if (i < N && j < N && i != j) {
            double v = J[i * N + j];
            double r = rint(v * scale);
            q = (int)r;
            if (i < j) { err += fabs(r * inv_scale - v); wq += (unsigned long long)(q < 0 ? -(long long)q : (long long)q); }
        }
        tab->Jq[idx] = q;
    }
    for (int i = tid; i < 64; i += blockDim.x) {
        int q = 0;
        if (i < N) {
            double v = FIELD_TERM_SIGN * h[i];                 // the one place the field sign convention enters the grid
            double r = rint(v * scale);
            q = (int)r;
            err += fabs(r * inv_scale - v);
            wq += (unsigned long long)(q < 0 ? -(long long)q : (long long)q);
        }
        tab->hq[i] = q;
    }
    s_red[tid] = err;
    if (wq) atomicAdd(&s_wq, wq);
    __syncthreads();
    for (int s = STAGE_THREADS / 2; s > 0; s >>= 1) {
        if (tid < s) s_red[tid] += s_red[tid + s];
        __syncthreads();
    }
    if (tid == 0) {
        double eps = s_red[0] + extra_eps_rel * W;     // extra: rounding done before staging (qubo_lowest)
        int exact = (eps == 0.0);
        int band = 0;
        if (!exact) {
            eps *= (1.0 + 1e-9);                               // rounding of the error sum itself
            double b = ceil(ldexp(2.0 * eps, p)) + 1.0;        // 2 epsilon in grid units, rounded up
            band = (b < 1.0e9) ? (int)b : 1000000000;
        }
        ctrl->status = ISING_OK;
        ctrl->p = p;
        ctrl->exact = exact;
        ctrl->band = band;
        ctrl->epsilon = eps;
        ctrl->W = W;
        // histogram of candidate energies (walk.cuh): HIST_FINE bins of 2^hist_shift grid units over [-Wq, +Wq]
        const long long Wq = (long long)s_wq;
        int hs = 0;
        while (((2 * Wq) >> hs) >= (long long)HIST_FINE) ++hs;
        ctrl->Wq = Wq;
        ctrl->hist_shift = hs;
        ctrl->count = 0;
        ctrl->kept = 0;
        ctrl->tau = tau_pack(TAU_INF, QC_NONE);
        ctrl->band_overflow = 0;
        ctrl->pool_overflow = 0;
        ctrl->next_unit = 0ull;
        ctrl->done_configs = 0ull;
        ctrl->count2 = 0;
        ctrl->final_state = 0;
        ctrl->eS = 0;
        ctrl->n_sure = 0;
        ctrl->blocks_done = 0;
        ctrl->hits = 0ull;
        ctrl->false_hits = 0ull;
        ctrl->z_steps = 0ull;
        ctrl->z_flagged = 0ull;
    }
    __syncthreads();                       // Jq, hq (global, written by this block) and Ctrl are complete
    build_tables(tab, ctrl, N);
}

// Tables of the QUBO form relative to the base state (see file header). Runs at the end of stage_kernel (one block);
// thread-per-entry loops.
__device__ void build_tables(Tables* __restrict__ tab, Ctrl* __restrict__ ctrl, int N)
{
    const int tid = threadIdx.x;
    const int* Jq = tab->Jq;
    auto Jat = [&](int i, int j) -> int { return (i < N && j < N) ? Jq[i * 64 + j] : 0; };

    for (int idx = tid; idx < NMID * NLO; idx += blockDim.x) {
        int mid = idx / NLO, lo = idx % NLO, acc = 0;
        for (int i = 0; i < LL; ++i) if (lo >> i & 1)
            for (int j = 0; j < LM; ++j) if (mid >> j & 1) acc += Jat(i, LL + j);
        tab->C[idx] = -4 * acc;
    }
    for (int lo = tid; lo < NLO; lo += blockDim.x) {
        int acc = 0;
        for (int i = 0; i < LL; ++i) if (lo >> i & 1)
            for (int j = i + 1; j < LL; ++j) if (lo >> j & 1) acc += Jat(i, j);
        tab->QL[lo] = -4 * acc;
    }
    for (int mid = tid; mid < NMID; mid += blockDim.x) {
        int acc = 0;
        for (int i = 0; i < LM; ++i) if (mid >> i & 1)
            for (int j = i + 1; j < LM; ++j) if (mid >> j & 1) acc += Jat(LL + i, LL + j);
        tab->QM[mid] = -4 * acc;
    }
    for (int idx = tid; idx < LW_MAX * 2 * NLO; idx += blockDim.x) {
        int k = idx / (2 * NLO), sb = (idx / NLO) & 1, lo = idx % NLO, acc = 0;
        for (int i = 0; i < LL; ++i) if (lo >> i & 1) acc += Jat(i, LOWBITS + k);
        tab->DV[idx] = (sb ? -4 : 4) * acc;
    }
    for (int idx = tid; idx < LW_MAX * 2 * NMID; idx += blockDim.x) {
        int k = idx / (2 * NMID), sb = (idx / NMID) & 1, mid = idx % NMID, acc = 0;
        for (int j = 0; j < LM; ++j) if (mid >> j & 1) acc += Jat(LL + j, LOWBITS + k);
        tab->DU[idx] = (sb ? -4 : 4) * acc;
    }
    for (int t = tid; t < (1 << LW_MAX); t += blockDim.x) {
        int v = 0;
        if (t > 0) {
            int k = __ffs(t) - 1;
            int gnew = t ^ (t >> 1);
            int sgn = (gnew >> k & 1) ? 1 : -1;
            int R = gnew & ~(1 << k);
            int acc = 0;
            for (int j = 0; j < LW_MAX; ++j) if (R >> j & 1) acc += Jat(LOWBITS + k, LOWBITS + j);
            v = -sgn * 4 * acc;
        }
        tab->DW[t] = v;
    }

    // ---- packed 16-bit screening tables (enumerate16.cu). One 16-bit unit = 2^s grid units; every entry is
    // floored, so V16 + C16 + U16 <= (V + C + U) / 2^s: a rigorous lower bound of the block energy.
    // Range: |Phi_i| <= R_i = |hq_i| + sum_j |Jq_ij| for every state, hence
    //   |V| <= BV = max|QL| + 2 sum_{i in lo} R_i,  |U| <= BU = max|QM| + 2 sum_{i in mid} R_i,  |C| <= BC = max|C|.
    // A quantised entry is off by less than 1 unit, a walked table by less than 1 + LW_MAX units (one floor per
    // set walk bit). s is the smallest shift for which no 16-bit lane can wrap (see enumerate16.cu header):
    // Every packed half is stored with an offset that makes it non-negative (so that packed words can be added with
    // plain 32-bit adds): V + bV, C + cC, U + cU with
    //   cC = (BC >> s) + 2,  cU = (BU >> s) + 2 + LW_MAX,  bV = (BV >> s) + 2 + LW_MAX + cC   (register set b holds
    //   V + C[16][.], hence the extra cC);  the largest half a sum can reach is 2 (bV + cC + cU) <= 65535.
    __shared__ int s_shift, s_cC;
    __shared__ unsigned long long s_BV, s_BU, s_BC;
    if (tid == 0) { s_BV = 0ull; s_BU = 0ull; s_BC = 0ull; }
    __syncthreads();                                   // QL, QM, C above are complete
    {
        unsigned long long m = 0ull;
        for (int x = tid; x < NMID * NLO; x += blockDim.x) { const long long v = tab->C[x]; const unsigned long long a = (unsigned long long)(v < 0 ? -v : v); if (a > m) m = a; }
        if (m) atomicMax(&s_BC, m);
        if (tid < NLO) { const long long v = tab->QL[tid]; atomicMax(&s_BV, (unsigned long long)(v < 0 ? -v : v)); }
        if (tid < NMID) { const long long v = tab->QM[tid]; atomicMax(&s_BU, (unsigned long long)(v < 0 ? -v : v)); }
    }
    __syncthreads();
    // R_i = |hq_i| + sum_j |Jq_ij| for the ten low spins, one warp each
    if (tid < 32 * LOWBITS) {
        const int i = tid >> 5, lane = tid & 31;
        unsigned long long R = 0ull;
        if (i < N) {
            for (int j = lane; j < N; j += 32) { const long long v = Jq[i * 64 + j]; R += (unsigned long long)(v < 0 ? -v : v); }
            if (lane == 0) { const long long v = tab->hq[i]; R += (unsigned long long)(v < 0 ? -v : v); }
        }
        if (R) atomicAdd(i < LL ? &s_BV : &s_BU, 2ull * R);
    }
    __syncthreads();
    if (tid == 0) {
        const long long BV = (long long)s_BV, BU = (long long)s_BU, BC = (long long)s_BC;
        int s = 0;
        long long cC = 0, cU = 0, bV = 0;
        for (; s < 40; ++s) {
            cC = (BC >> s) + 2;
            cU = (BU >> s) + 2 + LW_MAX;
            bV = (BV >> s) + 2 + LW_MAX + cC;
            if (2 * (bV + cC + cU) <= 65535) break;
        }
        s_shift = s;
        s_cC = (int)cC;
        tab->shift16 = s;
        tab->cU16 = (int)cU;
        tab->cC16 = (int)cC;
        tab->bV16 = (int)bV;
        ctrl->shift16 = s;
    }
    __syncthreads();
    const int s16 = s_shift;
    // pairing: the two halves of a packed word differ in mid bit 3 (spin LL + 3); u = 0..15 runs over the other four
    // mid bits, mid0(u) = (u & 7) | ((u >> 3) << 4). Rows u < 8 have mid bit 4 clear, rows u >= 8 have it set.
    for (int idx = tid; idx < (NMID / 2) * NLO; idx += blockDim.x) {
        const int u = idx / NLO, lo = idx % NLO;
        const int m0 = (u & 7) | ((u >> 3) << 4);
        const int a = (tab->C[m0 * NLO + lo] >> s16) + s_cC, b = (tab->C[(m0 | 8) * NLO + lo] >> s16) + s_cC;
        tab->Cp[idx] = (unsigned)a + ((unsigned)b << 16);        // both halves non-negative
    }
    for (int idx = tid; idx < LW_MAX * NLO; idx += blockDim.x) {
        const int k = idx / NLO, lo = idx % NLO;
        int acc = 0;
        for (int i = 0; i < LL; ++i) if (lo >> i & 1) acc += Jat(i, LOWBITS + k);
        const int d = (-4 * acc) >> s16;               // = DV[k][1][lo] >> s : the bit turns on
        tab->DVp[(k * 2 + 1) * NLO + lo] = (unsigned)(d * 65537);
        tab->DVp[(k * 2 + 0) * NLO + lo] = (unsigned)(-d * 65537);
    }
    for (int idx = tid; idx < LW_MAX * (NMID / 2); idx += blockDim.x) {
        const int k = idx / (NMID / 2), r = idx % (NMID / 2);
        const int m0 = (r & 7) | ((r >> 3) << 4), m1 = m0 | 8;
        int acc0 = 0, acc1 = 0;
        for (int j = 0; j < LM; ++j) {
            if (m0 >> j & 1) acc0 += Jat(LL + j, LOWBITS + k);
            if (m1 >> j & 1) acc1 += Jat(LL + j, LOWBITS + k);
        }
        const int d0 = (-4 * acc0) >> s16, d1 = (-4 * acc1) >> s16;
        const int D = d0 + 65536 * d1;                 // integer sum: halves never wrap (biased, non-negative)
        tab->DUp[(k * 2 + 1) * (NMID / 2) + r] = (unsigned)D;
        tab->DUp[(k * 2 + 0) * (NMID / 2) + r] = (unsigned)(-D);
    }
}

void launch_stage(const double* J, const double* h, int N, Tables* tab, Ctrl* ctrl, unsigned* hist, cudaStream_t st,
                  double extra_eps_rel)
{
    stage_kernel<<<1, STAGE_THREADS, 0, st>>>(J, h, N, tab, ctrl, hist, extra_eps_rel);
}

// QUBO -> Ising, eqs. (2),(3) inverted: J = a/4, h_i = b_i/2 + sum_j a_ij/4.
__global__ void qubo_to_ising_kernel(const double* __restrict__ a, const double* __restrict__ b, int N,
                                     double* __restrict__ J, double* __restrict__ h)
{
    for (int idx = threadIdx.x; idx < N * N; idx += blockDim.x) J[idx] = 0.25 * a[idx];
    for (int i = threadIdx.x; i < N; i += blockDim.x) {
        double acc = 0.0;
        for (int j = 0; j < N; ++j) if (j != i) acc += a[i * N + j];
        h[i] = FIELD_TERM_SIGN * (0.5 * b[i] + 0.25 * acc);
    }
}
void launch_qubo_to_ising(const double* a, const double* b, int N, double* J, double* h, cudaStream_t st)
{
    qubo_to_ising_kernel<<<1, 256, 0, st>>>(a, b, N, J, h);
}

}  // namespace ising
