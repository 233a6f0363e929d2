// k_inject.cu -- step S5 (selection term, eq. 12-13) and step S6 (combine, eq. 3).
//
//   S5  one CTA per (lambda, chunk of detected injections).  Both variants of the lambda's mass table (fp32 cubics,
//       2 x 32 KB) are brought into shared memory by one TMA bulk copy -- the injections' source masses are scattered
//       over the whole table -- and the chunk's packed records are streamed through it with coalesced 128-bit loads
//       (the set is sorted in d_L, so a warp's rows of the z(ln d_L) table are one or two L1-resident lines).  CTAs in
//       flight share a chunk (lambda is the fast grid index), so the records come from L2.  Per (injection, lambda):
//       log2 s_j = log2[p_m psi u / J / p_draw] via the same sample_eval() as the events (the injection table's r
//       column carries psi u / J); z_j > z_cat_max gives s_j = 0 (R6; the comparison is made on hi + lo pairs).
//       Chunks that span <= 0.9 in ln d_L (all of them for a dense set: it is sorted) replace the table rows by
//       chunk-local polynomials fitted per (chunk, lambda) (fit_polys / poly_sample, chim_internal.cuh).
//       s_j is widened to fp64 through the exponent field; per-CTA fp64 partial sums {sum s, sum s^2}, combined in a
//       fixed order by S6 (deterministic).
//   S6  log L = sum_i log I_i - N_e log xi, N_eff (eq. 13), flags.
#include "chim_internal.cuh"

namespace chim {

#ifndef CHIM_S5_UNROLL
#define CHIM_S5_UNROLL 2
#endif
constexpr int kS5Unroll = CHIM_S5_UNROLL;
constexpr int kInjThreads = 256;
constexpr int kInjChunkBlocks = 64;       // blocks of kInjThreads injections per chunk (chim_api.cu: kInjChunk = 16384)

struct InjSmem {
    LamConst L;
    double red[2 * (kInjThreads / 32)];
    unsigned long long mbar;
    alignas(16) float poly[4 * kPolyN];   // chunk-local polynomials (chim_internal.cuh)
};

__device__ __forceinline__ uint32_t inj_smem_u32(const void* p) { return (uint32_t)__cvta_generic_to_shared(p); }

// kDbg: the diagnostic instantiation also writes every s_j (chim_debug_injection_weights)
template <bool kDbg>
__global__ void __launch_bounds__(kInjThreads, 3) k_inject(InjKernelParams P) {
    extern __shared__ __align__(128) unsigned char smem_raw[];
    InjSmem& S = *reinterpret_cast<InjSmem*>(smem_raw);
    MassRow* mass_s = reinterpret_cast<MassRow*>(smem_raw + ((sizeof(InjSmem) + 127) / 128) * 128);
    const int tid = threadIdx.x, lane = tid & 31, wid = tid >> 5;
    const int l = blockIdx.x % P.n_lambda, chunk = blockIdx.x / P.n_lambda;
    const int64_t j0 = (int64_t)chunk * P.chunk, j1 = min(j0 + (int64_t)P.chunk, P.inj.n_det);
    const int nw = sizeof(LamConst) / 4;
    const MassRow* mtab = P.mtab + (size_t)l * 2 * (P.n_mass + 2);
    if (tid == 0) {   // TMA: the whole mass table of this lambda (both variants are contiguous)
        const uint32_t mb = inj_smem_u32(&S.mbar), bytes = 2u * (uint32_t)(P.n_mass + 2) * (uint32_t)sizeof(MassRow);
        asm volatile("mbarrier.init.shared::cta.b64 [%0], 1;" ::"r"(mb) : "memory");
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
        asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(mb), "r"(bytes) : "memory");
        asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];" ::"r"(inj_smem_u32(mass_s)),
                     "l"(mtab), "r"(bytes), "r"(mb)
                     : "memory");
    }
    for (int i = tid; i < nw; i += kInjThreads)
        reinterpret_cast<uint32_t*>(&S.L)[i] = reinterpret_cast<const uint32_t*>(P.Lc + l)[i];
    __syncthreads();   // publishes S.L and the initialised barrier
    {
        uint32_t ok;
        do {
            asm volatile("{\n .reg .pred p;\n mbarrier.try_wait.parity.shared::cta.b64 p, [%1], 0;\n selp.u32 %0, 1, 0, p;\n}"
                         : "=r"(ok)
                         : "r"(inj_smem_u32(&S.mbar))
                         : "memory");
        } while (!ok);
    }
    MassLookup M;
    M.g = mtab;
    M.s = mass_s;
    M.lo = 0;
    M.cap = P.n_mass + 2;
    M.n_mass = P.n_mass;
    const LamConst& L = S.L;
    const LamF& F = L.F;
    double acc[2] = {0.0, 0.0};
    double chunk_scale = 1.0;     // 2^(rounding residual of the chunk polynomial's constant term), applied to the chunk's sums in fp64
    int oor = 0;
    const double tk_h = P.inj.tk_h[chunk], tk_c = P.inj.tk_c[chunk];
    const bool use_poly = L.flags == 0 && tk_h > 0.0 && tk_c + tk_h < L.tkmax_inj;   // (block-uniform)
    if (use_poly) {
        // chunk-local polynomials: the chunk's injections span a narrow range of ln d_L; z is taken relative to z_cat_max, so the
        // support cut of R6 is the sign of the polynomial.  The chunk is ordered by m2d (chim_init_injections): warps whose
        // secondaries all lie below m_low (5-25 % of a reference set that starts at 5 Msun) leave after the 1/(1+z) polynomial,
        // and the warps above the smoothing window skip its three MUFU (vote).  For chunks narrower than 0.2 in ln d_L the
        // Madau-Dickinson turnover is part of the fitted polynomial r (k_polyfit; slot 26 of the record says so).
        const float* pr = P.poly + ((size_t)l * P.n_chunks + chunk) * (4 * kPolyN);
        PolyCoef C;
        {
            const float4* q = reinterpret_cast<const float4*>(pr);
            float4 v[7];
#pragma unroll
            for (int k = 0; k < 7; ++k) v[k] = __ldg(q + k);
            const float* f = reinterpret_cast<const float*>(v);
#pragma unroll
            for (int n = 0; n < kPolyN; ++n) C.zr[n] = pack2(f[2 * n], f[2 * n + 1]);
#pragma unroll
            for (int n = 0; n < kPolyN - 1; ++n) C.ua[n] = pack2(f[2 * kPolyN + 2 * n], f[2 * kPolyN + 2 * n + 1]);
        }
        const bool turn_folded = __float_as_int(__ldg(pr + 26)) != 0;
        chunk_scale = exp2((double)__ldg(pr + 27));
        const float4* pa = P.inj.prec_a + j0;                // padded to whole chunks with copies of the chunk's last injection
        const float2* pb = P.inj.prec_b + j0;
        const int n = (int)(j1 - j0), n32 = (n + 31) & ~31;
        const float tm_hi = F.tm_max;
        // the blocks of 256 injections whose secondaries ALL lie below m_low (the chunk is ordered by m2d; blk_m2d holds the
        // largest m2d of every block, 1/(1+z) is largest at the near end t = -1) contribute nothing (R15): the sweep starts
        // behind them
        int k0 = 0;
        {
            float amax = 0.f, sg = 1.f;
#pragma unroll
            for (int k = 0; k < kPolyN - 1; ++k) {
                float un, an;
                unpack2(C.ua[k], un, an);
                amax = fmaf(sg, an, amax);
                sg = -sg;
            }
            amax *= 1.0f + 1e-5f;
            const float* bm = P.inj.blk_m2d + (size_t)chunk * (kInjChunkBlocks);
            const int nblk = (n + kInjThreads - 1) / kInjThreads;
            // (one round trip: lane L looks at blocks L and L + 32; the block maxima increase with the block index)
            const unsigned lo = __ballot_sync(0xffffffffu, !(__ldg(bm + lane) * amax < F.mlow_hi));
            const unsigned hi = __ballot_sync(0xffffffffu, !(__ldg(bm + 32 + lane) * amax < F.mlow_hi));
            k0 = lo ? __ffs(lo) - 1 : (hi ? 32 + __ffs(hi) - 1 : kInjChunkBlocks);
            k0 = max(0, min(k0, nblk - 1));
        }
        // kDbg: s_j as a double through the exponent field, every one written out.  Production: fp32 sums of s_j / 2^ref and its
        // square per THREAD, ref the thread's own running reference -- raised (and the sums rescaled) whenever a weight exceeds
        // it by more than 2^40, a rare thread-local branch; the thread's sums become doubles once, at the end.  Weights more than
        // 2^126 below the reference are flushed: less than 2^-86 of the thread's largest.  8 instructions per injection less
        // than the fp64 accumulation.
#define CHIM_INJ_TAIL(TURN, MID, JJ)                                                                                  \
        {                                                                                                             \
            const float l2w = poly_tail<TURN, false>(F, F.gk2_inj, F.cpsi_inj, M, MID, nullptr);                      \
            if (kDbg) {                                                                                               \
                const double s = ((MID).zc <= 0.f && (JJ) < n) ? ex2_to_double(l2w) : 0.0;                            \
                acc[0] += s;                                                                                          \
                acc[1] = fma(s, s, acc[1]);                                                                           \
                if ((JJ) < n) P.dbg_s[P.inj.perm[j0 + (JJ)]] = s * P.dbg_scale * chunk_scale;                         \
            } else {                                                                                                  \
                const float lw = ((MID).zc <= 0.f && (JJ) < n) ? l2w : -INFINITY;                                     \
                if (lw > ref + 40.f) {   /* (NaN never enters: it fails the comparison and poisons the sums below) */  \
                    const float dn = ex2f(ref - lw);                                                                  \
                    f0 *= dn;                                                                                         \
                    f1 *= dn * dn;                                                                                    \
                    ref = lw;                                                                                         \
                }                                                                                                     \
                const float s = ex2f(lw - ref);                                                                       \
                f0 += s;                                                                                              \
                f1 = fmaf(s, s, f1);                                                                                  \
            }                                                                                                         \
        }
        // two blocks per iteration: both heads (they consume the records), the records of the next two blocks as one group of
        // loads, then both tails (chim_internal.cuh: poly_head / poly_tail)
#define CHIM_INJ_SWEEP(TURN)                                                                                          \
        {                                                                                                             \
            int j = tid + k0 * kInjThreads;                                                                           \
            const float4* pa_t = pa + j;                                                                              \
            const float2* pb_t = pb + j;                                                                              \
            PRec R0 = ldg_stream_prec(pa_t, pb_t), R1 = ldg_stream_prec(pa_t + kInjThreads, pb_t + kInjThreads);      \
            _Pragma("unroll 1") for (; j + kInjThreads < n32; j += 2 * kInjThreads) {                                 \
                PolyMid M0, M1;                                                                                       \
                poly_head(F, C, R0.A, R0.B, M, 1.0f, tm_hi, M0);                                                      \
                poly_head(F, C, R1.A, R1.B, M, 1.0f, tm_hi, M1);                                                      \
                ldg_stream_pair_after(R0, R1, pa_t + 2 * kInjThreads, pb_t + 2 * kInjThreads, pa_t + 3 * kInjThreads, \
                                      pb_t + 3 * kInjThreads, M0.rb, M1.rb);                                          \
                CHIM_INJ_TAIL(TURN, M0, j)                                                                            \
                CHIM_INJ_TAIL(TURN, M1, j + kInjThreads)                                                              \
                pa_t += 2 * kInjThreads;                                                                              \
                pb_t += 2 * kInjThreads;                                                                              \
            }                                                                                                         \
            if (j < n32) {                                                                                            \
                PolyMid M0;                                                                                           \
                poly_head(F, C, R0.A, R0.B, M, 1.0f, tm_hi, M0);                                                      \
                CHIM_INJ_TAIL(TURN, M0, j)                                                                            \
            }                                                                                                         \
        }
        if (kDbg)
            for (int j = tid; j < min(k0 * kInjThreads, n); j += kInjThreads) P.dbg_s[P.inj.perm[j0 + j]] = 0.0;
        float ref = -1e30f, f0 = 0.f, f1 = 0.f;
        if (turn_folded) CHIM_INJ_SWEEP(false)
        else CHIM_INJ_SWEEP(true)
        if (!kDbg) {   // the thread's sums on the absolute scale: s = 2^ref x relative weight
            const double sc = ex2_to_double(ref);                      // (ref never raised: f0 = f1 = 0, sc = 0)
            acc[0] = (double)f0 * sc;
            acc[1] = (double)f1 * sc * sc;
        }
#undef CHIM_INJ_SWEEP
#undef CHIM_INJ_TAIL
    } else if (L.flags == 0) {
        const float4* rows = reinterpret_cast<const float4*>(P.tab + (size_t)l * P.tab_rows);
        const int64_t j1w = j0 + ((j1 - j0 + 31) & ~(int64_t)31);    // whole warps stay in the loop (sample_eval votes)
        Rec R = ldg_stream_rec(P.inj.rec + 2 * min(j0 + tid, j1 - 1));
#pragma unroll(kS5Unroll)
        for (int64_t j = j0 + tid; j < j1w; j += kInjThreads) {
            const float4 A = R.A, Bq = R.B;
            if (j + kInjThreads < j1w) R = ldg_stream_rec(P.inj.rec + 2 * min(j + kInjThreads, j1 - 1));   // one iteration ahead
            const int k = __float_as_int(A.x);           // in [1, K]: clamped when the records were packed
            const float t = A.y;
            const bool in_range = ((float)k + t) <= F.tkmax_inj;
            const float4* r = rows + 4 * (size_t)k;
            const float4 q0 = __ldg(r), q1 = __ldg(r + 1), q2 = __ldg(r + 2), q3 = __ldg(r + 3);
            float zc, l2w;
            sample_eval(F, q0, q1, q2, q3, t, F.zcat_hi, F.zcat_lo, A.z, 0.f, A.w, 0.f, Bq.x, Bq.y, Bq.z, M, in_range, zc, l2w);
            oor |= (int)!in_range;
            const double s = (zc <= 0.f && j < j1) ? ex2_to_double(l2w) : 0.0;   // support of the selection-term z density (R6)
            acc[0] += s;
            acc[1] = fma(s, s, acc[1]);
            if (kDbg && j < j1) P.dbg_s[P.inj.perm[j]] = s * P.dbg_scale;
        }
    }
    acc[0] = warp_sum(acc[0]);
    acc[1] = warp_sum(acc[1]);
    if (lane == 0) { S.red[wid] = acc[0]; S.red[kInjThreads / 32 + wid] = acc[1]; }
    oor = __syncthreads_or(oor);   // also publishes S.red
    if (tid == 0) {
        double a = 0.0, b = 0.0;
#pragma unroll
        for (int k = 0; k < kInjThreads / 32; ++k) { a += S.red[k]; b += S.red[kInjThreads / 32 + k]; }
        P.partial[(size_t)chunk * P.n_lambda + l] = make_double2(a * chunk_scale, b * chunk_scale * chunk_scale);
        if (oor) atomicOr(P.flags + l, CHIM_FLAG_TABLE_RANGE);
    }
}

size_t inject_smem_bytes(int n_mass) {
    return ((sizeof(InjSmem) + 127) / 128) * 128 + 2 * sizeof(MassRow) * (size_t)(n_mass + 2);
}

cudaError_t launch_inject(const InjKernelParams& P, int n_blocks, cudaStream_t st) {
    if (n_blocks <= 0) return cudaSuccess;
    size_t smem = inject_smem_bytes(P.n_mass);
    auto kern = P.dbg_s ? k_inject<true> : k_inject<false>;
    cudaError_t e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    if (e != cudaSuccess) return e;
    kern<<<(unsigned)((long long)n_blocks * P.n_lambda), kInjThreads, smem, st>>>(P);
    return cudaGetLastError();
}

// ---- S6 ------------------------------------------------------------------------------------------------
constexpr int kCombThreads = 128;

__global__ void __launch_bounds__(kCombThreads) k_combine(CombineParams P) {
    __shared__ double red[3 * (kCombThreads / 32)];
    const int l = blockIdx.x, tid = threadIdx.x;
    const uint32_t lflags = P.Lc[l].flags;
    uint32_t fl = lflags | P.flags_in[l];
    double v[3] = {0.0, 0.0, 0.0};   // sum log I, sum s, sum s^2
    int n_ninf = 0, n_nan = 0;
    if (P.n_groups > 0) {   // many-1d: I_g = sum_k F_k I_k over the pixels of event g, in log space (eq. 14's pixel sum)
        fl &= ~CHIM_FLAG_EVENT_ZERO;             // raised per sub-event by k_events; here an empty pixel is not an empty event
        if (P.out_event_logI)
            for (int i = tid; i < P.n_events; i += kCombThreads)
                P.out_event_logI[(size_t)l * P.n_events + i] = P.logI[(size_t)l * P.n_events + i];
        for (int g = tid; g < P.n_groups; g += kCombThreads) {
            // R24: a pixel whose bandwidth is undefined (log I_k = NaN; k_events raised BW_DEGENERATE) is left out of the sum;
            // an event none of whose pixels has I_k > 0 is NaN if a pixel was left out, else empty
            const int64_t k0 = P.group_off[g], k1 = P.group_off[g + 1];
            double mx = -INFINITY;
            bool nan = false;
            for (int64_t k = k0; k < k1; ++k) {
                const double x = P.logI[(size_t)l * P.n_events + k] + P.ln_factor[k];
                if (isnan(x)) nan = true;
                else mx = fmax(mx, x);
            }
            if (mx == -INFINITY) {
                if (nan) n_nan = 1;
                else n_ninf = 1;
            } else {
                double acc = 0.0;
                for (int64_t k = k0; k < k1; ++k) {
                    const double x = P.logI[(size_t)l * P.n_events + k] + P.ln_factor[k];
                    if (!isnan(x)) acc += exp(x - mx);
                }
                v[0] += mx + log(acc);
            }
        }
    } else
    for (int i = tid; i < P.n_events; i += kCombThreads) {
        double x = P.logI[(size_t)l * P.n_events + i];
        if (P.out_event_logI) P.out_event_logI[(size_t)l * P.n_events + i] = x;
        if (isnan(x)) n_nan = 1;
        else if (isinf(x)) n_ninf = 1;
        else v[0] += x;
    }
    if (P.n_det > 0)
        for (int b = tid; b < P.n_inj_blocks; b += kCombThreads) {
            double2 p = P.partial[(size_t)b * P.n_lambda + l];
            v[1] += p.x;
            v[2] += p.y;
        }
    block_sum<kCombThreads, 3>(v, red);
    n_nan = __syncthreads_or(n_nan);
    n_ninf = __syncthreads_or(n_ninf);
    if (tid != 0) return;
    const int n_obs = (P.n_groups > 0) ? P.n_groups : P.n_events;   // N_obs of eq. 3
    if (P.n_groups > 0 && n_ninf && !n_nan) fl |= CHIM_FLAG_EVENT_ZERO;
    double total = n_nan ? NAN : (n_ninf ? -INFINITY : v[0]);
    double logxi = 0.0, neff = NAN;
    if (lflags) { total = NAN; logxi = NAN; }
    else if (P.n_det > 0) {
        double xi = v[1] / P.n_inj_total;
        neff = v[1] * v[1] / (v[2] - v[1] * v[1] / P.n_inj_total);
        if (!(xi > 0.0)) { fl |= CHIM_FLAG_XI_ZERO; logxi = NAN; total = NAN; }
        else {
            logxi = log(xi) + P.inj_ln_shift;
            if (neff < P.neff_factor * n_obs) fl |= CHIM_FLAG_NEFF_LOW;   // R8: report only
            total -= n_obs * logxi;
        }
    }
    P.out_loglike[l] = total;
    if (P.out_logxi) P.out_logxi[l] = logxi;
    if (P.out_neff) P.out_neff[l] = neff;
    if (P.out_flags) P.out_flags[l] = fl;
}

cudaError_t launch_combine(const CombineParams& P, cudaStream_t st) {
    if (P.n_lambda <= 0) return cudaSuccess;
    k_combine<<<P.n_lambda, kCombThreads, 0, st>>>(P);
    return cudaGetLastError();
}

}  // namespace chim
