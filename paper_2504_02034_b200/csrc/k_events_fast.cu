// k_events_fast.cu -- steps S2 + S3 + S4 for the regular case, one CTA per (event, lambda): narrow distance posterior
// (event-local polynomials), equally spaced redshift grid, Gaussian kernel in the local-expansion
// form, placement ON_SAMPLES.  Everything else -- wide events, other kernels / forms / placements,
// binning, diagnostics -- and every unit this kernel finds outside its reach (no or few effective samples, every supported
// secondary deep in the smoothing window, a bandwidth the expansion cannot take: DESIGN.md R21) is left to k_events: the unit
// is appended to a work list that k_events processes in the same batch call.
//
// Structure (what differs from k_events): between its five barriers the warps are independent.
//   prologue: every global load of the unit in one batch; q_g and the mass-table rows arrive by TMA bulk copies.   [barrier 1]
//   S2   warp w owns a contiguous chunk of the (d_L-sorted) samples and makes ONE sweep over it: the 26 polynomial
//        coefficients in registers, the records two blocks ahead (heads of two samples, one group of record loads, the two
//        tails), weights relative to a chunk reference found in the first block, moments about the centre of the event's
//        d_L range; it leaves chunk statistics {reference log2 w, sum w, sum w^2, sum w u, sum w u^2}.               [barrier 2]
//        Every warp combines the chunk statistics (lane c takes chunk c; sums of positive terms, fp32) and derives bandwidth
//        and expansion geometry redundantly; the psi table and the first sample of every box are found once per CTA
//        (one thread per entry).                                                                                  [barrier 3]
//   S3   the expansion coefficients of the boxes are built in groups of five boxes over the warps.                 [barrier 4]
//        Then every warp evaluates its own chunk of samples with per-sample box records from shared memory (no box search,
//        balanced), S4 folded in (q_g carries the trapezoid weights).                                             [barrier 5]
//        Warp 0 adds the per-warp sums and writes log I.
#include "chim_internal.cuh"

namespace chim {

constexpr int kFastBlocks8 = 3;      // resident CTAs per SM the eight-warp class is compiled for (80 registers)
// (threads per CTA kFT = 32 kFW, warps = sample chunks kFW: template parameter of the kernel, 8 or 4)
constexpr int kFPass = kFastPass;    // samples per warp pass (4 per lane)
constexpr int kFLeP = 12;            // terms of the local expansion
constexpr int kFMaxBox = 96;         // boxes per event
constexpr int kFBoxRec = 16;          // floats per box in shared memory: 12 coefficients, the box centre, 3 unused (64-byte records)
constexpr int kFGroup = 5;            // boxes whose coefficients one warp builds at a time
constexpr float kFMaxW = 1.3f;       // largest box width in units of sqrt(2) h
// largest half-width of the psi table: FastEventParams::max_d (grid points; ~60 on the spectroscopic, ~240 on the 4096-point
// photometric grids); 2 max_d zeros on both sides of the staged q_g: the coefficient build reads g_b +- d unchecked
constexpr int kFMassStage = 384;     // mass-table rows staged per variant (>= events_mass_stage_rows: k_polyfit sizes the slice)

template <int kFW>
struct FastSmem {
    unsigned long long mbar_mass, mbar_q;
    float4 win;                      // the window constants of S(m2) {win_lo, win_hi, two_dl2e, d2l2e} (read inside the vote only)
    float c_ref[kFW];                // per chunk: the reference log2 w of its weights (-inf: no weighted sample)
    float c_mom[kFW][4];             // sum w, sum w^2, sum w u, sum w u^2 with w relative to c_ref, u = z - z_mid
    float c_f[kFW];                  // 2^(c_ref - largest c_ref): chunk-relative weights -> one scale for the event
    double c_sum[kFW];               // per warp: sum_j w_j A_j over its boxes, relative to the event's largest weight
};

__host__ __device__ inline size_t fast_nz4(size_t nz) { return (nz + 3) / 4 * 4; }
__host__ __device__ inline size_t fast_aux_bytes(int max_d) {
    const size_t a = 2 * (size_t)kFMassStage * sizeof(MassRow);
    const size_t b = 4 * ((size_t)kFLeP * (size_t)(max_d + 1) + (size_t)kFBoxRec * (size_t)kFMaxBox);
    return a > b ? a : b;
}
size_t events_fast_smem_bytes(int max_ns, int max_nz, int warps, int max_d) {
    const size_t head = warps == 8 ? sizeof(FastSmem<8>) : (warps == 4 ? sizeof(FastSmem<4>) : sizeof(FastSmem<2>));
    return ((head + 127) / 128) * 128 + sizeof(float2) * (size_t)warps * fast_chunk(max_ns, warps) +
           sizeof(float) * (4 * (size_t)max_d + fast_nz4((size_t)max_nz)) + fast_aux_bytes(max_d);
}

template <int kFW, int kFMaxD>
__global__ void __launch_bounds__(32 * kFW, kFW == 8 ? kFastBlocks8 : (kFW == 4 ? 6 : 12)) k_events_fast(FastEventParams P) {
    constexpr int kFT = 32 * kFW;
    extern __shared__ __align__(128) unsigned char smem_raw[];
    FastSmem<kFW>& S = *reinterpret_cast<FastSmem<kFW>*>(smem_raw);
    constexpr int kFQPad = 2 * kFMaxD;                                  // (kFMaxD = the cap of the launch's class)
    float2* zw = reinterpret_cast<float2*>(smem_raw + ((sizeof(FastSmem<kFW>) + 127) / 128) * 128);   // (z_j - z0, log2 w_j -> w_j)
    float* qs = reinterpret_cast<float*>(zw + (size_t)kFW * fast_chunk(P.max_ns, kFW));          // [kFQPad | nz4 | kFQPad]
    unsigned char* aux = reinterpret_cast<unsigned char*>(qs + 2 * (size_t)kFQPad + fast_nz4((size_t)P.ev.max_nz));
    MassRow* mass_s = reinterpret_cast<MassRow*>(aux);                  // S2: both variants of the event's slice of the mass table
    float* psi = reinterpret_cast<float*>(aux);                         // S3: psi table [(D+1) x 12] ...
    float* Bc = psi + (size_t)kFLeP * (kFMaxD + 1);                     // ... and the box records [box][16]: 12 expansion coefficients, centre
    const int tid = threadIdx.x, lane = tid & 31, wid = tid >> 5;

    const int l = blockIdx.x % P.n_lambda;                              // lambda fastest: CTAs in flight share an event
    const int ev = P.fast_events[blockIdx.x / P.n_lambda];
    // Everything the unit needs from global memory is requested here in one batch, before the first branch that depends on any
    // of it (three dependent round trips -- event, these, records / mass rows -- instead of six): offsets, the per-lambda
    // constants, the 28-float record of k_polyfit (26 polynomial coefficients and the slice of the mass table to stage).
    const LamConst* Lg = P.Lc + l;
    const float* pr = P.poly + ((size_t)l * P.ev.n_events + ev) * (4 * kPolyN);
    float4 v[7];
    {
        const float4* q = reinterpret_cast<const float4*>(pr);
#pragma unroll
        for (int k = 0; k < 7; ++k) v[k] = __ldg(q + k);
    }
    LamF F;
    load_lamf_hot(F, &Lg->F);
    const uint32_t lflags = __ldg(&Lg->flags);
    const double tkmax = __ldg(&Lg->tkmax_ev);
    const int64_t s0 = __ldg(P.ev.sample_off + ev), s1 = __ldg(P.ev.sample_off + ev + 1);
    const int64_t g0 = __ldg(P.ev.grid_off + ev), g1 = __ldg(P.ev.grid_off + ev + 1);
    const int64_t p0 = __ldg(P.ev.poly_off + ev), q0off = __ldg(P.ev.q4_off + ev);
    const double tk_h = __ldg(P.ev.tk_h + ev), tk_c = __ldg(P.ev.tk_c + ev);
    const int ns = (int)(s1 - s0), nz = (int)(g1 - g0);
    double* out = P.logI + (size_t)l * P.ev.n_events + ev;
    if (lflags) {   // invalid lambda: NaN
        if (tid == 0) *out = NAN;
        return;
    }
    // the event-local polynomials exist (k_polyfit) iff the whole d_L range of the event lies inside the table
    int mlo = 0, nr = 0;
    if (tk_h > 0.0 && tk_c + tk_h < tkmax) {
        mlo = __float_as_int(v[6].z);
        nr = __float_as_int(v[6].w);                // > 0: every mass-table row the event can address fits the stage
    }
    // (bit 31 of a work-list entry: the unit needs the careful sweep of k_events -- it then skips its own fast one)
#define CHIM_FAST_HANDOVER(CAREFUL)                                             \
    do {                                                                        \
        if (tid == 0) {                                                         \
            const unsigned k_ = atomicAdd(P.work_count, 1u);                    \
            P.worklist[k_] = ((uint32_t)l * (uint32_t)P.ev.n_events + (uint32_t)ev) | ((CAREFUL) ? 0x80000000u : 0u); \
        }                                                                       \
        return;                                                                 \
    } while (0)
    if (nr <= 0 || nr > kFMassStage) CHIM_FAST_HANDOVER(false);

    const size_t nz4 = fast_nz4((size_t)nz);
    const MassRow* mtab = P.mtab + (size_t)l * 2 * (P.n_mass + 2);
    if (tid == 0) {
        S.win = make_float4(F.win_lo, F.win_hi, F.two_dl2e, F.d2l2e);
        mbar_init(&S.mbar_mass, 1);
        mbar_init(&S.mbar_q, 1);
        const uint32_t mbytes = (uint32_t)nr * (uint32_t)sizeof(MassRow);
        mbar_expect_tx(&S.mbar_mass, 2 * mbytes);
        bulk_g2s(mass_s, mtab + mlo, mbytes, &S.mbar_mass);
        bulk_g2s(mass_s + kFMassStage, mtab + (P.n_mass + 2) + mlo, mbytes, &S.mbar_mass);
        const uint32_t qbytes = (uint32_t)nz4 * 4u;
        mbar_expect_tx(&S.mbar_q, qbytes);
        bulk_g2s(qs + kFQPad, P.ev.qn4 + q0off, qbytes, &S.mbar_q);
    }
    for (int i = tid; i < kFQPad; i += kFT) {
        qs[i] = 0.f;
        qs[kFQPad + nz4 + i] = 0.f;
    }
    // per-thread copies of the 26 polynomial coefficients, paired for the packed FMAs
    PolyCoef Cf;
    {
        const float* f = reinterpret_cast<const float*>(v);
#pragma unroll
        for (int n = 0; n < kPolyN; ++n) Cf.zr[n] = pack2(f[2 * n], f[2 * n + 1]);
#pragma unroll
        for (int n = 0; n < kPolyN - 1; ++n) Cf.ua[n] = pack2(f[2 * kPolyN + 2 * n], f[2 * kPolyN + 2 * n + 1]);
    }
    // the warp's chunk [c0, c1) of the (d_L-sorted) samples; its first two blocks of records are requested here, ahead of the
    // barrier and of the wait for the mass rows
    const int C = fast_chunk(ns, kFW);
    const int c0 = wid * C, c1 = min(c0 + C, ns);
    const float4* pa = P.ev.prec_a + p0;
    const float2* pb = P.ev.prec_b + p0;
    PRec R0, R1;
    {
        const int jf = min(c0, ns - 1) + lane;                          // (warps beyond the event read its last block and drop it)
        R0 = ldg_stream_prec(pa + jf, pb + jf);
        R1 = ldg_stream_prec(pa + jf + 32, pb + jf + 32);
    }
    __syncthreads();                                                    // (1) the barriers are initialised
    MassLookup M;
    M.g = mtab;
    M.s = mass_s;
    M.lo = mlo;
    M.cap = kFMassStage;
    M.n_mass = P.n_mass;
    const float tm_lo = fmaxf(1.0f, (float)mlo), tm_hi = fminf(F.tm_max, (float)(mlo + nr) - 0.01f);

    // ---- S2 on the warp's chunk, one sweep: (z_j - z0, w_j) pairs to shared memory and the chunk's moments ---------------------------
    // w_j = 2^(log2 w_j - ref), ref = the largest log2 w of the first block of the chunk that has a weighted sample (any reference
    // within ~2^100 of the chunk's largest weight serves; one that is not shows up as inf/NaN moments and the unit is handed over).
    // Moments about z_mid = z at the centre of the event's d_L range (the constant term of the z polynomial): sums of positive
    // terms; the variance is taken about the weighted mean afterwards.
    float ref = 0.f;
    bool ref_unset = true;
    float m0 = 0.f, m1 = 0.f, m2 = 0.f, m3 = 0.f;
    float zmid, r0_unused;
    unpack2(Cf.zr[0], zmid, r0_unused);
    mbar_wait(&S.mbar_mass, 0);
    if (c0 < ns) {
        // running pointers (records, results) and a block count instead of an index: fewer live registers in the loop
        int nblk = (c1 - c0) >> 5;                                      // whole blocks of 32 samples
        const bool ragged = ((c1 - c0) & 31) != 0;
        const float4* pa_t = pa + c0 + lane;
        const float2* pb_t = pb + c0 + lane;
        float2* zw_t = zw + c0 + lane;
#define CHIM_FAST_TAIL(MID, OFF, IN, SEARCH)                                                                      \
        {                                                                                                         \
            const float l2w_ = poly_tail<true, true>(F, F.gk2, F.cpsi, M, MID, &S.win);                           \
            const float lw_ = (IN) ? l2w_ : -INFINITY;                                                            \
            if ((SEARCH) && ref_unset) {   /* (warp-uniform) */                                                   \
                float b_ = lw_;                                                                                   \
                _Pragma("unroll") for (int o = 16; o > 0; o >>= 1) b_ = fmaxf(b_, __shfl_xor_sync(0xffffffffu, b_, o)); \
                if (b_ > -INFINITY) {                                                                             \
                    ref = b_;                                                                                     \
                    ref_unset = false;                                                                            \
                }                                                                                                 \
            }                                                                                                     \
            const float w_ = ex2f(lw_ - ref), u_ = (MID).zc - zmid, wu_ = w_ * u_;                                \
            m0 += w_;                                                                                             \
            m1 = fmaf(w_, w_, m1);                                                                                \
            m2 += wu_;                                                                                            \
            m3 = fmaf(wu_, u_, m3);                                                                               \
            zw_t[OFF] = make_float2((MID).zc, w_);                                                                \
        }
        // Two samples per iteration: both heads (they consume the records), the records of the next two blocks as one group of
        // loads -- a full tail phase and the next heads away from their use -- then both tails.  The record arrays carry a spare
        // tail, so the loads are unconditional.
#define CHIM_FAST_PAIR(SEARCH)                                                                                    \
        {                                                                                                         \
            PolyMid M0, M1;                                                                                       \
            poly_head(F, Cf, R0.A, R0.B, M, tm_lo, tm_hi, M0);                                                    \
            poly_head(F, Cf, R1.A, R1.B, M, tm_lo, tm_hi, M1);                                                    \
            ldg_stream_pair_after(R0, R1, pa_t + 64, pb_t + 64, pa_t + 96, pb_t + 96, M0.rb, M1.rb);              \
            CHIM_FAST_TAIL(M0, 0, true, SEARCH)                                                                   \
            CHIM_FAST_TAIL(M1, 32, true, SEARCH)                                                                  \
            pa_t += 64;                                                                                           \
            pb_t += 64;                                                                                           \
            zw_t += 64;                                                                                           \
        }
        // the first loop runs until the chunk's reference is set (normally one iteration), the second is the plain one
#pragma unroll 1
        for (; nblk >= 2 && ref_unset; nblk -= 2) CHIM_FAST_PAIR(true)
#pragma unroll 1
        for (; nblk >= 2; nblk -= 2) CHIM_FAST_PAIR(false)
        // an odd block, then the ragged end of the event (records padded to whole warps with copies of the last sample:
        // poly_tail votes); the lanes beyond the event store that sample's redshift with weight 0 -- S3 reads the pair of the
        // last sample unmasked
        {
            PolyMid M0;
            if (nblk) {
                poly_head(F, Cf, R0.A, R0.B, M, tm_lo, tm_hi, M0);
                CHIM_FAST_TAIL(M0, 0, true, true)
                zw_t += 32;
                R0 = R1;
            }
            if (ragged) {
                poly_head(F, Cf, R0.A, R0.B, M, tm_lo, tm_hi, M0);
                CHIM_FAST_TAIL(M0, 0, (int)(zw_t - zw) < c1, true)
            }
        }
#undef CHIM_FAST_PAIR
#undef CHIM_FAST_TAIL
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) {
            m0 += __shfl_xor_sync(0xffffffffu, m0, o);
            m1 += __shfl_xor_sync(0xffffffffu, m1, o);
            m2 += __shfl_xor_sync(0xffffffffu, m2, o);
            m3 += __shfl_xor_sync(0xffffffffu, m3, o);
        }
        if (lane == 0) {
            S.c_ref[wid] = ref_unset ? -INFINITY : ref;
            S.c_mom[wid][0] = m0; S.c_mom[wid][1] = m1; S.c_mom[wid][2] = m2; S.c_mom[wid][3] = m3;
        }
    } else if (lane == 0) {
        S.c_ref[wid] = -INFINITY;
        S.c_mom[wid][0] = 0.f; S.c_mom[wid][1] = 0.f; S.c_mom[wid][2] = 0.f; S.c_mom[wid][3] = 0.f;
    }
    __syncthreads();                                                    // (2) chunk statistics and the samples are complete

    // ---- every warp: the event's moments from the eight chunks (lane c takes chunk c), bandwidth, expansion geometry -------------
    // fp32 throughout: all sums are sums of positive terms (the second moment is taken about the weighted mean in a second
    // step), n_eff >= neff_min (64; 24 for many-1d pixels) on this path, and dh/h = 1e-6 moves log I by ~5e-9
    const float cm = (lane < kFW) ? S.c_ref[lane] : -INFINITY;
    float gref = cm;
#pragma unroll
    for (int o = kFW / 2; o > 0; o >>= 1) gref = fmaxf(gref, __shfl_xor_sync(0xffffffffu, gref, o));
    gref = __shfl_sync(0xffffffffu, gref, 0);
    mbar_wait(&S.mbar_q, 0);                                            // q_g has landed (also: no copy in flight at any exit below)
    if (!(gref > -INFINITY)) CHIM_FAST_HANDOVER(true);                   // no weighted sample on this path: k_events decides
    const bool live = lane < kFW && cm > -INFINITY;
    const float f = live ? ex2f(cm - gref) : 0.f;                       // chunk-relative weights -> relative to the largest chunk reference
    const float wc = live ? S.c_mom[lane][0] : 0.f, qc = live ? S.c_mom[lane][1] : 0.f;
    const float bc = live ? S.c_mom[lane][2] : 0.f, ac = live ? S.c_mom[lane][3] : 0.f;
    if (wid == 0 && lane < kFW) S.c_f[lane] = f;
    float SW = f * wc, SQ = f * f * qc, SB = f * bc;
#pragma unroll
    for (int o = kFW / 2; o > 0; o >>= 1) {
        SW += __shfl_xor_sync(0xffffffffu, SW, o);
        SQ += __shfl_xor_sync(0xffffffffu, SQ, o);
        SB += __shfl_xor_sync(0xffffffffu, SB, o);
    }
    SW = __shfl_sync(0xffffffffu, SW, 0);
    SQ = __shfl_sync(0xffffffffu, SQ, 0);
    SB = __shfl_sync(0xffffffffu, SB, 0);
    const float de = -__fdividef(SB, SW);                                          // minus the weighted mean (relative to z_mid)
    float SA = f * fmaf(de, fmaf(de, wc, 2.f * bc), ac);                // sum w (u + de)^2 >= 0 per chunk
#pragma unroll
    for (int o = kFW / 2; o > 0; o >>= 1) SA += __shfl_xor_sync(0xffffffffu, SA, o);
    SA = __shfl_sync(0xffffffffu, SA, 0);
    const float s2 = __fdividef(SQ, SW * SW), neff = __fdividef(1.0f, s2);   // sum w^^2, Kish n_eff
    float h;   // (fast divisions and MUFU powers: dh/h = 1e-6 moves log I by ~5e-9)
    if (P.bw_rule == CHIM_BW_FIXED) {
        h = (float)__ldg(P.ev.fixed_bw + ev);
    } else {   // Scott on the weighted sample (R3, O7): sigma^2 = sum w^(z - zbar)^2 / (1 - sum w^^2), h = sigma n_eff^(-1/5)
        const float var = __fdividef(SA, SW * (1.0f - s2));
        h = (var > 0.f) ? sqrtf(var) * ex2f(0.2f * lg2f(s2)) : NAN;
    }
    // handed over: no bandwidth; few effective samples (fp32 weights, moments and the plain form of Scott's rule are good for
    // n_eff >> 1 only); every supported secondary deep in the smoothing window (m2' < ~0.3 sqrt(delta): d ln w = delta/m2'^2 x 1e-6)
    // the largest m2' of the event, bounded from below chunk by chunk: the chunk's largest m2d (packed at init) at the chunk's far
    // end, where 1/(1+z) is smallest (within 0.5 % of the exact value; the unit is handed over whenever the exact criterion would)
    float gmp2 = -INFINITY;
    if (lane < kFW) {
        const float2 ct = __ldg(P.ev.chunk_top + (size_t)ev * kFastWarps + lane);   // {largest m2d, t of the last sample} of chunk `lane`
        float un, a1;
        unpack2(Cf.ua[kPolyN - 2], un, a1);
#pragma unroll
        for (int n = kPolyN - 3; n >= 0; --n) {
            float an;
            unpack2(Cf.ua[n], un, an);
            a1 = fmaf(a1, ct.y, an);
        }
        gmp2 = fmaf(ct.x, a1, -F.mlow_hi);                               // (empty chunks: m2d = 0)
    }
#pragma unroll
    for (int o = kFW / 2; o > 0; o >>= 1) gmp2 = fmaxf(gmp2, __shfl_xor_sync(0xffffffffu, gmp2, o));
    gmp2 = __shfl_sync(0xffffffffu, gmp2, 0);
    const bool hand_careful = !(h > 0.f) || !isfinite(h) || !(neff >= P.neff_min) || gmp2 < 0.f || gmp2 * gmp2 < 0.1f * F.delta;
    bool hand = hand_careful;
    // local-expansion geometry: y = z'/(sqrt(2) h), boxes of m grid spacings centred on grid points
    const double udz = __ldg(P.ev.uni_dz + ev), zfirst = __ldg(P.ev.zc + g0);
    const float scy = 0.70710678118654752440f / h;
    const float dy = (float)(udz * (double)scy);
    const int m = max(1, (int)lrintf(__fdividef(1.0f, dy)));
    const float wbox = (float)m * dy, Ty = (float)P.cutoff * 0.70710678118654752440f;
    const float yfirst = (float)(zfirst * (double)scy), inv_w = __fdividef(1.0f, wbox);
    const float fb_lo = floorf((zw[0].x * scy - yfirst) * inv_w + 0.5f), fb_hi = floorf((zw[ns - 1].x * scy - yfirst) * inv_w + 0.5f);
    const float fD = ceilf(__fdividef(Ty + 0.5f * wbox, dy)) + 1.0f;
    hand = hand || !(wbox <= kFMaxW) || !(fb_hi - fb_lo < (float)kFMaxBox) || !(fabsf(fb_lo) < 1e6f) || !(fabsf(fb_hi) < 1e6f) ||
           !(fD <= (float)kFMaxD) || !(fabsf(fb_lo) * (float)m < 1e8f) || !(fabsf(fb_hi) * (float)m < 1e8f);
    if (hand) CHIM_FAST_HANDOVER(hand_careful);
    const int D = (int)fD, b_lo = (int)fb_lo, nbox = (int)(fb_hi - fb_lo) + 1;
    // once per CTA, one thread per entry: the psi table psi_n(d dy) = exp(-t^2) H_n(t)/n!, t = d dy, by the three-term recurrence
    for (int d = tid; d <= D; d += kFT) {
        const float t = (float)d * dy, t2 = 2.f * t;
        float p0v = ex2f(-t * t * 1.44269504088896341f), p1v = t2 * p0v;
        float* o = psi + (size_t)d * kFLeP;
        o[0] = p0v;
        o[1] = p1v;
#pragma unroll
        for (int n = 1; n < kFLeP - 1; ++n) {
            const float p2v = fmaf(t2, p1v, -2.f * p0v) * (1.0f / (float)(n + 1));
            o[n + 1] = p2v;
            p0v = p1v;
            p1v = p2v;
        }
    }
    __syncthreads();                                                    // (3) psi table (the staged mass rows are dead)

    // ---- S3, coefficients: groups of five consecutive boxes, group g built by warp g mod 8 -----------------------------------------
    // B_bn = sum_{|d| <= D} q_{g_b+d} psi_n(d dy): lane = (half of the d range, box of the group, quad of n); psi_n(-t) =
    // (-1)^n psi_n(t), so even n take (q_+ + q_-) psi_n and odd n (q_+ - q_-) psi_n -- the pairs (n, n+1) of a packed FMA
    {
        const int half = lane >= 15 ? 1 : 0, sub = lane - 15 * half, quad = sub % 3, bsub = sub / 3;
        const int Dh = D >> 1, d_lo = half ? Dh + 1 : 1, d_hi = half ? D : Dh;
        for (int base = kFGroup * wid; base < nbox; base += kFGroup * kFW) {
            const int bi = base + bsub;
            const bool valid = lane < 30 && bi < nbox;
            const int gc = (b_lo + (valid ? bi : 0)) * m;               // grid index of the box centre
            const bool reach = valid && gc > -D - 1 && gc < nz + D;     // else no grid point within the box's cut-off: B = 0
            const float* qp = qs + kFQPad + (reach ? gc : 0) + d_lo;
            const float* qm = qs + kFQPad + (reach ? gc : 0) - d_lo;
            const float4* pp = reinterpret_cast<const float4*>(psi) + quad + d_lo * (kFLeP / 4);
            f32x2 a01 = 0ull, a23 = 0ull;
            if (reach && !half) {   // d = 0: psi_odd(0) = 0
                const float q0 = qp[-d_lo];
                const float4 v = reinterpret_cast<const float4*>(psi)[quad];
                a01 = pack2(q0 * v.x, 0.f);
                a23 = pack2(q0 * v.z, 0.f);
            }
            int n = reach ? d_hi - d_lo + 1 : 0;
#pragma unroll 1
            for (; n >= 4; n -= 4) {
#pragma unroll
                for (int k = 0; k < 4; ++k) {
                    const float a = qp[k], b = qm[-k];
                    const float4 v = pp[k * (kFLeP / 4)];
                    const f32x2 qeo = pack2(a + b, a - b);
                    a01 = fma2(qeo, pack2(v.x, v.y), a01);
                    a23 = fma2(qeo, pack2(v.z, v.w), a23);
                }
                qp += 4;
                qm -= 4;
                pp += 4 * (kFLeP / 4);
            }
            for (; n > 0; --n) {
                const float a = *qp, b = *qm;
                const float4 v = *pp;
                const f32x2 qeo = pack2(a + b, a - b);
                a01 = fma2(qeo, pack2(v.x, v.y), a01);
                a23 = fma2(qeo, pack2(v.z, v.w), a23);
                ++qp;
                --qm;
                pp += kFLeP / 4;
            }
            float4 acc;
            unpack2(a01, acc.x, acc.y);
            unpack2(a23, acc.z, acc.w);
            acc.x += __shfl_down_sync(0xffffffffu, acc.x, 15);          // the two halves of the d range
            acc.y += __shfl_down_sync(0xffffffffu, acc.y, 15);
            acc.z += __shfl_down_sync(0xffffffffu, acc.z, 15);
            acc.w += __shfl_down_sync(0xffffffffu, acc.w, 15);
            if (valid && !half) {
                reinterpret_cast<float4*>(Bc + (size_t)bi * kFBoxRec)[quad] = acc;
                if (quad == 0) Bc[(size_t)bi * kFBoxRec + kFLeP] = fmaf((float)gc, dy, yfirst);   // the box centre c_b
            }
        }
    }
    __syncthreads();                                                    // (4) the box records are complete

    // ---- S3 + S4, evaluation: warp w on its own chunk of the samples (the one it wrote in S2: one weight scale per warp) --------------
    // per sample its box b = round((y - y_first)/w) - b_lo (any box whose centre is within ~w/2 serves; clamped to the boxes that
    // exist), the box record from shared memory (neighbouring lanes mostly share it: broadcast), s = y - c_b and one degree-11
    // polynomial; four samples per lane and pass (pairs jb, jb + 1 and jb + 64, jb + 65: 16-byte lane stride)
    double lsum = 0.0;
    if (c0 < ns) {
        const float kb = 0.5f - (float)b_lo - yfirst * inv_w;
        const int bmax = nbox - 1;
        const float4* B4 = reinterpret_cast<const float4*>(Bc);
        const int jsafe = (ns - 1) & ~1;                                // (slots beyond the chunk's last pair read that pair; their weights are masked)
        const int pend = c0 + ((c1 - c0 + kFPass - 1) / kFPass) * kFPass;
        for (int jb = c0 + 2 * lane; jb < pend; jb += kFPass) {
            const float4 ab = *reinterpret_cast<const float4*>(zw + min(jb, jsafe)), cd4 = *reinterpret_cast<const float4*>(zw + min(jb + 64, jsafe));
            const float zv[4] = {ab.x, ab.z, cd4.x, cd4.z};
            const float wv[4] = {ab.y, ab.w, cd4.y, cd4.w};
            float y[4], v[4];
#pragma unroll
            for (int r = 0; r < 4; ++r) y[r] = zv[r] * scy;
            // the samples are sorted: if the first and the last sample of the pass fall into the same box, all 128 do (dense
            // boxes: most passes) -- then the box record is read once, broadcast, and two samples share a packed FMA
            const int bf = min(max(__float2int_rd(fmaf(y[0], inv_w, kb)), 0), bmax), bl = min(max(__float2int_rd(fmaf(y[3], inv_w, kb)), 0), bmax);
            const int b_first = __shfl_sync(0xffffffffu, bf, 0), b_last = __shfl_sync(0xffffffffu, bl, 31);
            if (b_first == b_last) {
                const float4* bp = B4 + b_first * (kFBoxRec / 4);
                const float4 k0 = bp[0], k1 = bp[1], k2 = bp[2];
                const float cb = bp[3].x;
                const f32x2 s01 = pack2(y[0] - cb, y[1] - cb), s23 = pack2(y[2] - cb, y[3] - cb);
                f32x2 a01 = pack2(k2.w, k2.w), a23 = a01;
#define CHIM_LE_STEP(cf) { const f32x2 q_ = pack2(cf, cf); a01 = fma2(a01, s01, q_); a23 = fma2(a23, s23, q_); }
                CHIM_LE_STEP(k2.z) CHIM_LE_STEP(k2.y) CHIM_LE_STEP(k2.x)
                CHIM_LE_STEP(k1.w) CHIM_LE_STEP(k1.z) CHIM_LE_STEP(k1.y) CHIM_LE_STEP(k1.x)
                CHIM_LE_STEP(k0.w) CHIM_LE_STEP(k0.z) CHIM_LE_STEP(k0.y) CHIM_LE_STEP(k0.x)
#undef CHIM_LE_STEP
                unpack2(a01, v[0], v[1]);
                unpack2(a23, v[2], v[3]);
            } else {
#pragma unroll
                for (int r = 0; r < 4; ++r) {
                    const int b = (r == 0) ? bf : (r == 3) ? bl : min(max(__float2int_rd(fmaf(y[r], inv_w, kb)), 0), bmax);
                    const float4* bp = B4 + b * (kFBoxRec / 4);
                    const float4 k0 = bp[0], k1 = bp[1], k2 = bp[2];
                    const float sv = y[r] - bp[3].x;
                    float t = k2.w;
                    t = fmaf(t, sv, k2.z); t = fmaf(t, sv, k2.y); t = fmaf(t, sv, k2.x);
                    t = fmaf(t, sv, k1.w); t = fmaf(t, sv, k1.z); t = fmaf(t, sv, k1.y); t = fmaf(t, sv, k1.x);
                    t = fmaf(t, sv, k0.w); t = fmaf(t, sv, k0.z); t = fmaf(t, sv, k0.y); t = fmaf(t, sv, k0.x);
                    v[r] = t;
                }
            }
            float a = 0.f;
#pragma unroll
            for (int r = 0; r < 4; ++r) {
                const bool in = jb + (r & 1) + 64 * (r >> 1) < c1;
                a = fmaf(in ? wv[r] : 0.f, v[r], a);
            }
            lsum += (double)a;
        }
        lsum = warp_sum(lsum) * (double)S.c_f[wid];
    }
    if (lane == 0) S.c_sum[wid] = lsum;
    __syncthreads();                                                    // (4)
    if (tid == 0) {
        double tot = 0.0;
#pragma unroll
        for (int k = 0; k < kFW; ++k) tot += S.c_sum[k];                // fixed order: deterministic
        // K(z) = 1/(N_s h sqrt(2 pi)) sum_j w_j exp(..); the weights were divided by 2^gref, the prior and q_g scales factored out
        const double I = tot / ((double)ns * (double)h * 2.50662827463100050242);
        if (I > 0.0 && isfinite(I)) {
            *out = log(I) + (double)gref * 0.69314718055994530942 + __ldg(P.ln_shift + ev) + __ldg(P.ln_qscale + ev);
        } else {   // nothing within the cut-off (or not a number): k_events evaluates the unit in log space
            const unsigned k_ = atomicAdd(P.work_count, 1u);
            P.worklist[k_] = (uint32_t)l * (uint32_t)P.ev.n_events + (uint32_t)ev;
        }
    }
#undef CHIM_FAST_HANDOVER
}

template <int kFW, int kFMaxD>
static cudaError_t launch_fast_t(const FastEventParams& P, long long nb, size_t smem, cudaStream_t st) {
    cudaError_t e = cudaFuncSetAttribute(k_events_fast<kFW, kFMaxD>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    if (e != cudaSuccess) return e;
    k_events_fast<kFW, kFMaxD><<<(unsigned)nb, 32 * kFW, smem, st>>>(P);
    return cudaGetLastError();
}

// the instantiations fast_warps_for() / fast_max_d_for() (chim_internal.cuh) can ask for
cudaError_t launch_events_fast(const FastEventParams& P, int n_fast, cudaStream_t st) {
    const long long nb = (long long)P.n_lambda * n_fast;
    if (nb <= 0) return cudaSuccess;
    const int w = P.warps, d = P.max_d;
    const size_t smem = events_fast_smem_bytes(P.max_ns, P.ev.max_nz, w, d);
    if (w == 8 && d == 256) return launch_fast_t<8, 256>(P, nb, smem, st);
    if (w == 8 && d == 384) return launch_fast_t<8, 384>(P, nb, smem, st);
    if (w == 4 && d == 160) return launch_fast_t<4, 160>(P, nb, smem, st);
    if (w == 4 && d == 384) return launch_fast_t<4, 384>(P, nb, smem, st);
    if (w == 2 && d == 160) return launch_fast_t<2, 160>(P, nb, smem, st);
    if (w == 2 && d == 384) return launch_fast_t<2, 384>(P, nb, smem, st);
    return cudaErrorInvalidValue;
}

}  // namespace chim
