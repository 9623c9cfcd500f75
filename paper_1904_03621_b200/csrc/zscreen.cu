// zscreen.cu -- SURVEY.md section 8 rows a3 + a4 on the 5th-generation tensor cores (tcgen05 / TMEM): the threshold
// screen of a block of 2^14 configurations as ONE dense contraction.
//
// The block energies decompose exactly as in enumerate.cu (the QUBO form of eqs. (2),(3), around the
// thread's base state with the 14 block spins down):
//      E(lo, mid) = Eh - 2 sum_{i in lo} Phi_i - 2 sum_{j in mid} Phi_j + C'(lo, mid),
//      C'(lo, mid) = -4 sum_{a<b both set in lo u mid} Jq_ab        (per instance; lo = spins 0..6, mid = spins 7..13)
// "Does the block hold a configuration with E <= tauE?" is a (min,+) question. Its (+,x) image is the block's
// partition function at inverse temperature lambda (bits per grid unit):
//      Z = sum_{lo,mid} 2^(-lambda (E(lo,mid) - tauE))  >=  2^(-lambda (E_min - tauE)),
// so  E_min <= tauE  implies  Z >= 1, and a block with Z < 1 cannot hold a candidate: THE SCREEN CAN PRODUCE FALSE
// HITS, NEVER A MISS -- provided Z is not under-estimated by more than the margin kept below. Z factorises,
//      Z = 2^L  sum_mid u[mid]  ( sum_lo T[mid][lo] a[lo] ),   T[mid][lo] = 2^(-lambda C'(lo,mid) + t0)   (per instance)
//      a[lo]  = prod_{i in lo}  2^(2 lambda Phi_i) / (largest such product)        in (0, 1]     (per thread and step)
//      u[mid] = prod_{j in mid} 2^(2 lambda Phi_j) / (largest such product)        in (0, 1]
//      L      = lambda (tauE - Eh) - t0 + sum_i max(2 lambda Phi_i, 0)                             (log domain, fp32)
// and the inner sum over lo is a GEMM: D[thread][mid] = sum_lo A[thread][lo] T[mid][lo] with A = the a-vectors of the
// 128 threads of the CTA -- M = 128 (threads), N = 128 (mid), K = 128 (lo), bf16 inputs, fp32 accumulation in TMEM,
// 2 flop per configuration. Per step a thread generates its A row (192 multiplies, written as bf16 in the UMMA
// canonical layout), one elected thread issues 8 tcgen05.mma (K = 16 each), and every thread folds its own D row
// (tcgen05.ld) with the u factors: 254 multiply-adds for 2^14 configurations, against 2^13 packed add-mins in
// enumerate16.cu. A flagged block is formed exactly (int32) by the warp, 16 x 1024 configurations (walk.cuh
// form_block), so what reaches the pool is identical to the other kernels.
//
// Why the screen is rigorous (DESIGN.md section 6b has the full argument):
//   * all terms are positive, so rounding only perturbs Z relatively: T and a are rounded to bf16 (2^-9 each, to
//     nearest), the fp32 products inside the tensor core are exact, accumulation, the u-fold and the factor chain add
//     < 2^-11; in the log domain that is < 0.007 bits, and L itself is good to 1e-3 bits. The test flags a block
//     unless  log2(Z~) + L < -0.02 ;
//   * underflow: a term of a configuration with E <= tauE has  log2 a + log2 T + log2 u >= -L; with |log2 T| <= THETA
//     (lambda is chosen from the range of C') none of its partial products is below 2^-(L + THETA), so for
//     L <= L_SAFE = 126 - THETA - 8 it cannot underflow; blocks with L > L_SAFE are flagged unconditionally
//     (their crude bound is far below tauE: they almost always do hold a candidate);
//   * overflow cannot happen (a, u <= 1, T <= 2^THETA), and a NaN can only make the comparison fail, i.e. flag.
#include <cuda_bf16.h>

#include "walk.cuh"

namespace ising {

constexpr int Z_THREADS = 128;
constexpr unsigned Z_LBO = 128, Z_SBO = 2048;          // UMMA canonical K-major layout without swizzle (bytes)
constexpr float Z_THETA = 40.f;                        // half range of log2 T
constexpr float Z_L_SAFE = 126.f - Z_THETA - 8.f;
constexpr float Z_MARGIN = 0.02f;
// kind::f16 instruction descriptor: D fp32, A and B bf16, both K-major, N = 128, M = 128
constexpr unsigned Z_IDESC = (1u << 4) | (1u << 7) | (1u << 10) | ((unsigned)(128 >> 3) << 17) | ((unsigned)(128 >> 4) << 24);
constexpr int Z_SMEM_BYTES = 32768 + 32768;            // T table + A tile (dynamic shared memory)

__device__ __forceinline__ unsigned smem_u32(const void* p) { return (unsigned)__cvta_generic_to_shared(p); }

__device__ __forceinline__ unsigned long long umma_desc(unsigned saddr)
{
    return (unsigned long long)((saddr >> 4) & 0x3fffu) | ((unsigned long long)(Z_LBO >> 4) << 16) |
           ((unsigned long long)(Z_SBO >> 4) << 32) | (1ull << 46);         // version 1, no swizzle, base offset 0
}

__device__ __forceinline__ float ex2f(float x) { float r; asm("ex2.approx.ftz.f32 %0, %1;" : "=f"(r) : "f"(x)); return r; }
__device__ __forceinline__ float lg2f(float x) { float r; asm("lg2.approx.ftz.f32 %0, %1;" : "=f"(r) : "f"(x)); return r; }
__device__ __forceinline__ unsigned pack_bf16(float lo, float hi)
{
    unsigned r;
    asm("cvt.rn.bf16x2.f32 %0, %1, %2;" : "=r"(r) : "f"(hi), "f"(lo));     // d.hi = first source, d.lo = second
    return r;
}

// ---- per-instance tables of the screen: one block, after stage_kernel ----
__global__ void __launch_bounds__(1024) ztables_kernel(const Tables* __restrict__ tab, const Ctrl* __restrict__ ctrl,
                                                       ZTables* __restrict__ zt, int N)
{
    if (ctrl->status != 0) return;
    __shared__ int s_min, s_max;
    __shared__ float s_lambda, s_t0;
    const int tid = threadIdx.x;
    const int* __restrict__ Jq = tab->Jq;
    if (tid == 0) { s_min = 0x7fffffff; s_max = -0x7fffffff; }
    __syncthreads();
    int mn = 0x7fffffff, mx = -0x7fffffff;
    for (int x = tid; x < (1 << ZB); x += blockDim.x) {
        int acc = 0;
        for (int a = 0; a < ZB; ++a)
            if (x >> a & 1)
                for (int b = a + 1; b < ZB; ++b)
                    if (x >> b & 1) acc += Jq[a * 64 + b];              // rows/columns >= N are zero
        const int c = -4 * acc;
        zt->Cz[x] = c;
        mn = min(mn, c);
        mx = max(mx, c);
    }
    atomicMin(&s_min, mn);
    atomicMax(&s_max, mx);
    for (int idx = tid; idx < LW_MAX * 16; idx += blockDim.x) {
        const int k = idx >> 4, i = idx & 15;
        zt->DPhi[idx] = (i < ZB && ZB + k < 64) ? 2 * Jq[i * 64 + ZB + k] : 0;
    }
    for (int t = tid; t < (1 << LW_MAX); t += blockDim.x) {
        int v = 0;
        if (t > 0) {
            const int k = __ffs(t) - 1;
            const int gnew = t ^ (t >> 1);
            const int sgn = (gnew >> k & 1) ? 1 : -1;
            const int R = gnew & ~(1 << k);
            int acc = 0;
            for (int j = 0; j < LW_MAX; ++j)
                if ((R >> j & 1) && ZB + k < 64 && ZB + j < 64) acc += Jq[(ZB + k) * 64 + ZB + j];
            v = -sgn * 4 * acc;
        }
        zt->DWz[t] = v;
    }
    __syncthreads();
    if (tid == 0) {
        // lambda: the table spans 2 THETA bits; an instance without couplings inside the block gets a sharp screen
        const double range = (double)s_max - (double)s_min;
        double lam = range > 0.0 ? 2.0 * (double)Z_THETA / range : 16.0;
        if (lam > 16.0) lam = 16.0;
        s_lambda = (float)lam;
        s_t0 = (float)(lam * 0.5 * ((double)s_max + (double)s_min));
        zt->lambda = s_lambda;
        zt->t0 = s_t0;
        zt->cmin = s_min;
        zt->cmax = s_max;
    }
    __syncthreads();
    const double lam = (double)s_lambda, t0 = (double)s_t0;
    unsigned short* Tb = reinterpret_cast<unsigned short*>(zt->Tb);
    for (int x = tid; x < (1 << ZB); x += blockDim.x) {
        const int lo = x & 127, mid = x >> 7;
        const double e = -lam * (double)zt->Cz[x] + t0;                  // |e| <= THETA (+ rounding of lambda, t0)
        const __nv_bfloat16 v = __float2bfloat16_rn((float)exp2(e));
        // canonical layout of the B operand: row = mid (N index), column = lo (K index)
        const unsigned off = (unsigned)(mid >> 3) * Z_SBO + (unsigned)(lo >> 3) * Z_LBO + (unsigned)(mid & 7) * 16u + (unsigned)(lo & 7) * 2u;
        Tb[off >> 1] = __bfloat16_as_ushort(v);
    }
}

// ---- the screen kernel: one CTA of 128 threads per unit of 2^(21 + Lw) configurations ----
__global__ void __launch_bounds__(Z_THREADS)
zwalk_kernel(const Tables* __restrict__ tab, const ZTables* __restrict__ zt, Ctrl* __restrict__ ctrl,
             Entry* __restrict__ pool, unsigned* __restrict__ hist, const __grid_constant__ Plan plan)
{
    extern __shared__ __align__(1024) unsigned char zsmem[];
    unsigned char* sT = zsmem;                       // 32 KB: B operand (the instance table)
    unsigned char* sA = zsmem + 32768;               // 32 KB: A operand (one row per thread)
    __shared__ __align__(8) unsigned long long mbar;
    __shared__ unsigned s_tmem;
    __shared__ unsigned long long s_unit;
    __shared__ int sDWz[1 << LW_MAX];
    __shared__ __align__(16) int sDPhi[LW_MAX * 16];
    __shared__ int sPhiW[LW_MAX][Z_THREADS];
    __shared__ int sPhiB[Z_THREADS / 32][64];

    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    if (ctrl->status != 0) return;
    // ---- take a unit ----
    if (tid == 0) s_unit = atomicAdd(&ctrl->next_unit, 1ull);
    for (int i = tid; i < 2048; i += Z_THREADS) reinterpret_cast<uint4*>(sT)[i] = zt->Tb[i];
    for (int i = tid; i < (1 << LW_MAX); i += Z_THREADS) sDWz[i] = zt->DWz[i];
    for (int i = tid; i < LW_MAX * 16; i += Z_THREADS) sDPhi[i] = zt->DPhi[i];
    if (tid == 0) {
        asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" :: "r"(smem_u32(&mbar)), "r"(1));
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    __syncthreads();
    const unsigned long long u = s_unit;
    if (u >= plan.total_units) return;
    int s = 0;
    while (s + 1 < plan.nseg && u >= plan.seg[s].first_unit + plan.seg[s].n_units) ++s;
    const int unit_bits = plan.seg[s].unit_bits;
    const int Lw = unit_bits - (ZB + 7);
    const int nlow = ZB + Lw;
    const unsigned long long qU = plan.seg[s].q0 + ((u - plan.seg[s].first_unit) << unit_bits);
    if (tid == 0) {
        const unsigned long long need = plan.seg[s].need_done;
        while (ld_relaxed_u64(&ctrl->done_configs) < need) {
            if (ld_relaxed_u32(&ctrl->pool_overflow)) break;
            __nanosleep(100);
        }
    }
    __syncwarp();
    if (warp == 0) {
        asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], %1;" :: "r"(smem_u32(&s_tmem)), "r"(128));
        asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;");
    }
    asm volatile("fence.proxy.async.shared::cta;" ::: "memory");          // the table copy is read by the tensor core
    asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory");
    __syncthreads();
    asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
    const unsigned tmem = s_tmem;
    const bool dead = ld_relaxed_u32(&ctrl->pool_overflow) != 0u;         // the run is void: only release TMEM

    const int N = plan.N;
    const int* __restrict__ Jq = tab->Jq;
    const float lambda = zt->lambda, t0 = zt->t0;
    unsigned long long flagged = 0ull;

    if (!dead) {
        // ---- a2: base state. Warp: Phi_i(qW), E(qW) for the warp's first state; lane: its 5 lane bits on top ----
        const unsigned long long qW = qU + ((unsigned long long)warp << (nlow + 5));
        int plo, phi;
        const int EW = warp_fields(tab, N, qW, lane, plo, phi);
        sPhiB[warp][lane] = plo;
        sPhiB[warp][lane + 32] = phi;
        __syncwarp();
        int Phi[ZB];
        int PhiW[LW_MAX];
#pragma unroll
        for (int i = 0; i < ZB; ++i) Phi[i] = sPhiB[warp][i];
#pragma unroll
        for (int i = 0; i < LW_MAX; ++i) PhiW[i] = (i < Lw) ? sPhiB[warp][ZB + i] : 0;
        int Eh = EW;
        for (int j = 0; j < 5 && nlow + j < N; ++j) {
            const bool fl = (lane >> j) & 1;
            const int a = nlow + j;
            const int* col = Jq + a * 64;
#pragma unroll
            for (int i = 0; i < ZB; ++i) Phi[i] += fl ? 2 * col[i] : 0;
#pragma unroll
            for (int i = 0; i < LW_MAX; ++i) PhiW[i] += (fl && i < Lw) ? 2 * col[ZB + i] : 0;
            int e = -2 * sPhiB[warp][a];
            for (int jj = 0; jj < j; ++jj)
                if ((lane >> jj) & 1) e -= 4 * col[nlow + jj];
            Eh += fl ? e : 0;
        }
#pragma unroll
        for (int i = 0; i < LW_MAX; ++i) sPhiW[i][tid] = PhiW[i];

        unsigned long long tau = ld_relaxed_u64(&ctrl->tau);
        int tauE = tau_energy(tau);
        unsigned parity = 0;
        const float two_lambda = 2.f * lambda;
        unsigned char* myrow = sA + (unsigned)(tid >> 3) * Z_SBO + (unsigned)(tid & 7) * 16u;
        const unsigned nsteps = 1u << Lw;

        for (unsigned t = 0; t < nsteps; ++t) {
            // ---- per-spin factors: bit set multiplies the weight by 2^y, y = 2 lambda Phi; normalised so that the
            //      larger of the two factors of a spin is exactly 1 ----
            float r0[ZB], r1[ZB];
            float Lp = lambda * (float)(tauE - Eh) - t0;
#pragma unroll
            for (int i = 0; i < ZB; ++i) {
                const float y = two_lambda * (float)Phi[i];
                const float e = ex2f(-fabsf(y));
                r1[i] = y >= 0.f ? 1.f : e;
                r0[i] = y >= 0.f ? e : 1.f;
                Lp += fmaxf(y, 0.f);
            }
            // ---- A row: a[lo] = prod over the 7 lo spins, 128 values, bf16, canonical layout ----
            {
                float P[32];
                P[0] = r0[0]; P[1] = r1[0];
#pragma unroll
                for (int b = 1; b < 5; ++b) {
#pragma unroll
                    for (int j = (1 << b) - 1; j >= 0; --j) {
                        const float v = P[j];
                        P[j + (1 << b)] = v * r1[b];
                        P[j] = v * r0[b];
                    }
                }
#pragma unroll
                for (int c = 0; c < 4; ++c) {
                    const float f = ((c & 1) ? r1[5] : r0[5]) * ((c & 2) ? r1[6] : r0[6]);
#pragma unroll
                    for (int g = 0; g < 4; ++g) {
                        uint4 w;
                        w.x = pack_bf16(P[8 * g + 0] * f, P[8 * g + 1] * f);
                        w.y = pack_bf16(P[8 * g + 2] * f, P[8 * g + 3] * f);
                        w.z = pack_bf16(P[8 * g + 4] * f, P[8 * g + 5] * f);
                        w.w = pack_bf16(P[8 * g + 6] * f, P[8 * g + 7] * f);
                        *reinterpret_cast<uint4*>(myrow + (unsigned)(4 * c + g) * Z_LBO) = w;   // k-chunk lo/8 = 4c + g
                    }
                }
            }
            asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
            asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory");
            __syncthreads();                 // every A row is written; every TMEM read of the previous step is done
            if (tid == 0) {
                asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
                const unsigned a0 = smem_u32(sA), b0 = smem_u32(sT);
#pragma unroll
                for (int ks = 0; ks < 8; ++ks) {
                    const unsigned long long da = umma_desc(a0 + (unsigned)ks * 2u * Z_LBO);
                    const unsigned long long db = umma_desc(b0 + (unsigned)ks * 2u * Z_LBO);
                    const unsigned acc = ks > 0 ? 1u : 0u;
                    asm volatile("{\n\t.reg .pred p;\n\tsetp.ne.b32 p, %4, 0;\n\t"
                                 "tcgen05.mma.cta_group::1.kind::f16 [%0], %1, %2, %3, p;\n\t}"
                                 :: "r"(tmem), "l"(da), "l"(db), "r"(Z_IDESC), "r"(acc) : "memory");
                }
                asm volatile("tcgen05.commit.cta_group::1.mbarrier::arrive::one.shared::cluster.b64 [%0];"
                             :: "r"(smem_u32(&mbar)) : "memory");
            }
            // ---- while the tensor core works: the Gray step that follows this block (walk bit k = ctz(t + 1)) ----
            const unsigned tn = t + 1 < nsteps ? t + 1 : 1u;
            const int k = __ffs(tn) - 1;
            const int sb = ((tn ^ (tn >> 1)) >> k) & 1;
            const int EhNext = Eh + sDWz[tn] + (sb ? -2 : 2) * sPhiW[k][tid];
            int dphi[16];
            {
                const int4* dp = reinterpret_cast<const int4*>(sDPhi + k * 16);
#pragma unroll
                for (int x = 0; x < 4; ++x) {
                    const int4 d = dp[x];
                    dphi[4 * x + 0] = d.x; dphi[4 * x + 1] = d.y; dphi[4 * x + 2] = d.z; dphi[4 * x + 3] = d.w;
                }
            }
            // ---- wait for the accumulator, fold this thread's row: R = sum_mid u[mid] D[mid] ----
            asm volatile("{\n\t.reg .pred P1;\n\tZWAIT_%=:\n\t"
                         "mbarrier.try_wait.parity.shared::cta.b64 P1, [%0], %1;\n\t"
                         "@P1 bra ZDONE_%=;\n\tbra ZWAIT_%=;\n\tZDONE_%=:\n\t}" :: "r"(smem_u32(&mbar)), "r"(parity) : "memory");
            parity ^= 1u;
            __syncwarp();
            asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
            float part[4];
#pragma unroll
            for (int c = 0; c < 4; ++c) {
                unsigned v[32];
                const unsigned taddr = tmem + ((unsigned)(warp * 32) << 16) + (unsigned)(c * 32);
                asm volatile("tcgen05.ld.sync.aligned.32x32b.x32.b32 "
                             "{%0, %1, %2, %3, %4, %5, %6, %7, %8, %9, %10, %11, %12, %13, %14, %15, "
                             "%16, %17, %18, %19, %20, %21, %22, %23, %24, %25, %26, %27, %28, %29, %30, %31}, [%32];"
                             : "=r"(v[0]), "=r"(v[1]), "=r"(v[2]), "=r"(v[3]), "=r"(v[4]), "=r"(v[5]), "=r"(v[6]), "=r"(v[7]),
                               "=r"(v[8]), "=r"(v[9]), "=r"(v[10]), "=r"(v[11]), "=r"(v[12]), "=r"(v[13]), "=r"(v[14]), "=r"(v[15]),
                               "=r"(v[16]), "=r"(v[17]), "=r"(v[18]), "=r"(v[19]), "=r"(v[20]), "=r"(v[21]), "=r"(v[22]), "=r"(v[23]),
                               "=r"(v[24]), "=r"(v[25]), "=r"(v[26]), "=r"(v[27]), "=r"(v[28]), "=r"(v[29]), "=r"(v[30]), "=r"(v[31])
                             : "r"(taddr) : "memory");
                asm volatile("tcgen05.wait::ld.sync.aligned;" ::: "memory");
                float x[32];
#pragma unroll
                for (int j = 0; j < 32; ++j) x[j] = __uint_as_float(v[j]);
                // mid bits 0..4 = spins 7..11: five butterfly stages
#pragma unroll
                for (int b = 0; b < 5; ++b) {
#pragma unroll
                    for (int j = 0; j < 32; j += (2 << b)) x[j] = fmaf(x[j + (1 << b)], r1[7 + b], x[j] * r0[7 + b]);
                }
                part[c] = x[0];
            }
            // mid bits 5, 6 = spins 12, 13
            const float h0 = fmaf(part[1], r1[12], part[0] * r0[12]);
            const float h1 = fmaf(part[3], r1[12], part[2] * r0[12]);
            const float R = fmaf(h1, r1[13], h0 * r0[13]);
            // ---- a4: flag unless the block provably holds no configuration with E <= tauE ----
            const bool clear = (lg2f(R) + Lp < -Z_MARGIN) && (Lp <= Z_L_SAFE);
            unsigned hits = __ballot_sync(0xffffffffu, !clear);
            flagged += __popc(hits);
            while (hits) {
                const int src = __ffs(hits) - 1;
                hits &= hits - 1;
                const unsigned gray = t ^ (t >> 1);
                const unsigned long long qh = qW + ((unsigned long long)src << nlow) + ((unsigned long long)gray << ZB);
#pragma unroll 1
                for (int sub = 0; sub < (1 << (ZB - LOWBITS)); ++sub) {
                    form_block<true>(tab, ctrl, pool, hist, plan, tab->C, qh + ((unsigned long long)sub << LOWBITS), 0, tau, lane);
                    tau = ld_relaxed_u64(&ctrl->tau);
                }
                tauE = tau_energy(tau);
            }
            // ---- move on to step t + 1 ----
            Eh = EhNext;
#pragma unroll
            for (int i = 0; i < ZB; ++i) Phi[i] += sb ? dphi[i] : -dphi[i];
            if ((t & 15u) == 15u) {
                tau = ld_relaxed_u64(&ctrl->tau);
                tauE = tau_energy(tau);
            }
        }
    }
    // ---- unit complete ----
    asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory");
    __syncthreads();
    if (lane == 0 && flagged) atomicAdd(&ctrl->z_flagged, flagged);
    if (tid == 0) {
        atomicAdd(&ctrl->z_steps, (unsigned long long)Z_THREADS << (dead ? 0 : Lw));
        __threadfence();
        if (!dead) atomicAdd(&ctrl->done_configs, 1ull << unit_bits);
    }
    __syncwarp();
    if (warp == 0) {
        asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
        asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, %1;" :: "r"(tmem), "r"(128));
    }
}

void launch_ztables(const Tables* tab, const Ctrl* ctrl, ZTables* zt, int N, cudaStream_t st)
{
    ztables_kernel<<<1, 1024, 0, st>>>(tab, ctrl, zt, N);
}

void launch_zwalk(const Tables* tab, const ZTables* zt, Ctrl* ctrl, Entry* pool, unsigned* hist, const Plan& plan,
                  cudaStream_t st)
{
    zwalk_kernel<<<(unsigned)plan.total_units, Z_THREADS, Z_SMEM_BYTES, st>>>(tab, zt, ctrl, pool, hist, plan);
}

void set_zscreen_attributes()
{
    cudaFuncSetAttribute(zwalk_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, Z_SMEM_BYTES);
}

}  // namespace ising
