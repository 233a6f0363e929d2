// k_events.cu -- steps S2 + S3 + S4 fused: one CTA per (event, lambda).
//
//   S2  per posterior sample: z_j from the per-lambda table, source masses, population weight w_j
//       (sample_weight, chim_internal.cuh), weighted moments -> Scott bandwidth h (R3), all in fp64.
//       z_j and w_j never leave shared memory.
//   S3+S4  I_i = sum_g q_g K(z_g) = (1/(N_s h sqrt(2 pi))) sum_j w_j A_j,  A_j = sum_g q_g exp(-(z_g - z_j)^2 / 2h^2),
//       q_g = p_gal(z_g) x trapezoid weight (eq. 19 evaluated on the grid, eq. 14).
//       Samples in lanes (4 per lane, 128 per warp pass, sorted in z), grid points streamed from shared memory;
//       a pass visits the grid band within t*h of its samples (R9).  Two formulations of the Gaussian:
//
//       power form (equally spaced grid): with x = z sqrt(log2(e)/2)/h, delta the grid spacing in
//       x, block start x_a, u = x_a - x_j and g = aB + b:
//           2^-(x_g - x_j)^2 = 2^(-u^2) * (2^(-2 delta u))^b * 2^(-b^2 delta^2)
//       so per block of B grid points  sum_b q_g E_gj = e0 * sum_b q'_b s^b  with q'_b = q_g 2^(-b^2 delta^2)
//       precomputed per CTA: a Horner polynomial in s -- ONE fp32 FMA per pair, issued as packed FFMA2 (two
//       samples per instruction), and two MUFU.EX2 (e0, s) per sample and block.  Exact up to fp32 rounding
//       (no recurrence across blocks: every block restarts from fresh exponentials).
//
//       direct form (any grid; also bandwidths below ~3 grid spacings, no cut-off, diagnostics):
//           A_j += q_g * ex2(-(x_g - x_j)^2)   FADD, FMUL, MUFU.EX2, FFMA per pair.
//
//   log I_i written per (lambda, event); block reductions in fp64.
#include "chim_internal.cuh"

namespace chim {

#ifndef CHIM_EV_THREADS
#define CHIM_EV_THREADS 256
#define CHIM_EV_BLOCKS 3
#endif
constexpr int kEvThreads = CHIM_EV_THREADS;   // 256 x 3 CTAs per SM measured faster than 384 x 2 and 512 x 1
constexpr int kPass = 128;               // samples per warp pass (4 per lane)
constexpr float kMaxBlockSpan = 4.8f;    // B * delta limit of the power form
constexpr float kMaxPowExp = 100.f;      // bound on log2 of the largest s^b inside a block (fp32 overflow guard)
constexpr int kMassStage = 384;          // mass-table rows staged per CTA during S2 (aliases the grid array of S3)

__device__ __forceinline__ float ex2_approx(float x) {
    float y;
    asm("ex2.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x));
    return y;
}
typedef unsigned long long f32x2;        // two packed floats (lo, hi) for the FFMA2 pipe
__device__ __forceinline__ f32x2 pack2(float lo, float hi) {
    f32x2 r;
    asm("mov.b64 %0, {%1, %2};" : "=l"(r) : "f"(lo), "f"(hi));
    return r;
}
__device__ __forceinline__ void unpack2(f32x2 v, float& lo, float& hi) {
    asm("mov.b64 {%0, %1}, %2;" : "=f"(lo), "=f"(hi) : "l"(v));
}
__device__ __forceinline__ f32x2 fma2(f32x2 a, f32x2 b, f32x2 c) {
    f32x2 d;
    asm("fma.rn.f32x2 %0, %1, %2, %3;" : "=l"(d) : "l"(a), "l"(b), "l"(c));
    return d;
}

// psi(z)/J(z) at a grid point for placement ON_GRID (paper eq. 14 literally); d_C from the global table.
__device__ double grid_factor(const LamConst& L, const double* __restrict__ dc, int n_nodes, double dz, double z) {
    double x = z / dz;
    int i = max(0, min((int)x, n_nodes - 2));
    double t = x - (double)i;
    double a0 = 1.0 + i * dz, a1e = 1.0 + (i + 1) * dz;
    double f0 = L.c_H0 * rsqrt(L.Om * a0 * a0 * a0 + 1.0 - L.Om) * dz;
    double f1 = L.c_H0 * rsqrt(L.Om * a1e * a1e * a1e + 1.0 - L.Om) * dz;
    double t2 = t * t, omt = 1.0 - t;
    double dcz = (1.0 + 2.0 * t) * omt * omt * dc[i] + t2 * (3.0 - 2.0 * t) * dc[i + 1] + t * omt * omt * f0 - t2 * omt * f1;
    double a = 1.0 + z, u = log1p(z);
    double fE = L.c_H0 * rsqrt(L.Om * a * a * a + 1.0 - L.Om);
    double xi = L.Xi0 + (1.0 - L.Xi0) * exp(-L.n * u);
    double dxi = -L.n * (1.0 - L.Xi0) * exp(-(L.n + 1.0) * u);
    double ddl = dxi * a * dcz + xi * (dcz + a * fE);
    double psi = exp(L.gamma * u) / (1.0 + exp(L.gk * (u - L.ln1pzp)));
    return psi / (a * a * a * fabs(ddl));
}

struct EvSmem {
    LamConst L;
    double red[4 * (kEvThreads / 32)];
    int pass_counter;
    int pad_;
};

__host__ __device__ inline size_t ev_ns_pad(size_t ns) { return (ns + kPass - 1) / kPass * kPass; }
__host__ __device__ inline size_t ev_nz_pad(size_t nz) { return (nz + 31) / 32 * 32; }
__host__ __device__ inline size_t ev_aux_bytes(size_t nz) {   // S2: staged mass rows; S3: (q', q') or (x_g, q_g) per grid point
    size_t a = sizeof(float2) * ev_nz_pad(nz), b = (size_t)kMassStage * 32;
    return a > b ? a : b;
}

// One block of B grid points for the 4 samples of a lane: tot_k += 2^(-u_k^2) * sum_b q'_b s_k^b (Horner, FFMA2).
template <int B>
__device__ __forceinline__ void power_block(const ulonglong2* __restrict__ qp, float xs, float cs, const float (&x)[4],
                                            f32x2& tot01, f32x2& tot23) {
    const float u0 = xs - x[0], u1 = xs - x[1], u2 = xs - x[2], u3 = xs - x[3];
    const f32x2 s01 = pack2(ex2_approx(cs * u0), ex2_approx(cs * u1));
    const f32x2 s23 = pack2(ex2_approx(cs * u2), ex2_approx(cs * u3));
    const f32x2 e01 = pack2(ex2_approx(-u0 * u0), ex2_approx(-u1 * u1));
    const f32x2 e23 = pack2(ex2_approx(-u2 * u2), ex2_approx(-u3 * u3));
    f32x2 a01 = 0ull, a23 = 0ull;     // (+0.f, +0.f)
#pragma unroll
    for (int i = B / 2 - 1; i >= 0; --i) {
        const ulonglong2 v = qp[i];   // {(q'_2i, q'_2i), (q'_2i+1, q'_2i+1)}
        a01 = fma2(a01, s01, v.y);
        a23 = fma2(a23, s23, v.y);
        a01 = fma2(a01, s01, v.x);
        a23 = fma2(a23, s23, v.x);
    }
    tot01 = fma2(e01, a01, tot01);
    tot23 = fma2(e23, a23, tot23);
}

template <int B>
__device__ __forceinline__ void power_pass(const float2* __restrict__ gq, int a_lo, int a_hi, float xfirst, float delta,
                                           const float (&x)[4], float (&A)[4]) {
    f32x2 tot01 = 0ull, tot23 = 0ull;
    const float cs = -2.f * delta;
#pragma unroll 1
    for (int a = a_lo; a <= a_hi; ++a) {
        const float xs = fmaf((float)(a * B), delta, xfirst);
        power_block<B>(reinterpret_cast<const ulonglong2*>(gq + a * B), xs, cs, x, tot01, tot23);
    }
    unpack2(tot01, A[0], A[1]);
    unpack2(tot23, A[2], A[3]);
}

// shared-memory layout after EvSmem: wbuf double[ns_pad] | zf float[ns_pad] | aux = gq float2[nz_pad] / staged mass rows
__global__ void __launch_bounds__(kEvThreads, CHIM_EV_BLOCKS) k_events(EventKernelParams P) {
    extern __shared__ __align__(16) unsigned char smem_raw[];
    EvSmem& S = *reinterpret_cast<EvSmem*>(smem_raw);
    double* wbuf = reinterpret_cast<double*>(smem_raw + ((sizeof(EvSmem) + 15) / 16) * 16);
    const size_t ns_pad = ev_ns_pad(P.ev.max_ns);
    float* zf = reinterpret_cast<float*>(wbuf + ns_pad);
    float2* gq = reinterpret_cast<float2*>(zf + ns_pad);
    const int tid = threadIdx.x, lane = tid & 31;

    int l, ev;
    if (P.dbg_event >= 0) { l = blockIdx.x; ev = P.dbg_event; }
    else { l = blockIdx.x % P.n_lambda; ev = blockIdx.x / P.n_lambda; }   // lambda fastest: CTAs in flight share an event
    const int64_t s0 = P.ev.sample_off[ev], g0 = P.ev.grid_off[ev];
    const int ns = (int)(P.ev.sample_off[ev + 1] - s0), nz = (int)(P.ev.grid_off[ev + 1] - g0);
    double* out = (P.dbg_event >= 0) ? P.logI + l : P.logI + (size_t)l * P.ev.n_events + ev;

    {   // stage the per-lambda constants in shared memory
        const int nw = sizeof(LamConst) / 4;
        const uint32_t* src = reinterpret_cast<const uint32_t*>(P.Lc + l);
        uint32_t* dst = reinterpret_cast<uint32_t*>(&S.L);
        for (int i = tid; i < nw; i += kEvThreads) dst[i] = src[i];
        if (tid == 0) S.pass_counter = 0;
    }
    __syncthreads();
    const LamConst& L = S.L;
    if (L.flags) {   // invalid lambda: NaN
        if (tid == 0) *out = NAN;
        return;
    }
    const Row* tab = P.tab + (size_t)l * P.tab_rows;
    const double z0 = P.ev.z0[ev];

    // ---- stage the mass-table rows this event can address: ln m1 = ln m1d - ln(1+z), z between the event's first and
    //      last (sorted) sample; rows outside the staged range fall back to global memory inside sample_weight ----------
    MassLookup M;
    M.g = P.mtab + (size_t)l * (P.n_mass + 2);
    M.n_mass = P.n_mass;
    M.cap = kMassStage;
    {
        double2* sA = reinterpret_cast<double2*>(gq);
        double2* sB = sA + kMassStage;
        const int ka = max(1, min((int)P.ev.recA[s0].x, P.tab_rows - 2)), kb = max(1, min((int)P.ev.recA[s0 + ns - 1].x, P.tab_rows - 2));
        const double u_lo = tab[ka].c[1][0], u_hi = tab[kb + 1].c[1][0];      // ln(1+z) at the bracketing nodes
        const int ma = max(1, min((int)fma(P.ev.lnm1_lo[ev] - u_hi - L.lm0, L.inv_dlm, 1.0), P.n_mass));
        const int mb = max(1, min((int)fma(P.ev.lnm1_hi[ev] - u_lo - L.lm0, L.inv_dlm, 1.0), P.n_mass));
        M.lo = ma + max(0, (mb - ma + 1 - kMassStage) / 2);                   // wider than the stage: keep the centre
        for (int i = tid; i < kMassStage; i += kEvThreads) {
            const int r = min(M.lo + i, P.n_mass + 1);
            double2 hi;
            const double2 lo = ldg256_lo(reinterpret_cast<const double*>(M.g + r), hi);
            sA[i] = lo;
            sB[i] = hi;
        }
        M.sA = sA;
        M.sB = sB;
    }
    __syncthreads();

    // ---- S2: weights + centred moments -----------------------------------------------------------------
    double mom[4] = {0.0, 0.0, 0.0, 0.0};   // sum w, sum w^2, sum w z', sum w z'^2
    int oor = 0;
    // software pipeline: the next sample's table coordinate is read one iteration ahead and its row prefetched to L1
    double2 A = (tid < ns) ? ldg_stream(P.ev.recA + s0 + tid) : make_double2(1.0, 1.0);
#pragma unroll 1
    for (int j = tid; j < ns; j += kEvThreads) {
        const double2 B = ldg_stream(P.ev.recB + s0 + j), C = ldg_stream(P.ev.recC + s0 + j);
        double2 An = A;
        if (j + kEvThreads < ns) {
            An = ldg_stream(P.ev.recA + s0 + j + kEvThreads);
            prefetch_l1(tab + max(1, min((int)An.x, P.tab_rows - 2)));
        }
        double z, w;
        bool o;
        sample_weight(L, tab, P.tab_rows, M, L.tkmax_ev, P.z_table_max, A.x, A.y, B.x, B.y, C.x, C.y, z, w, o);
        oor |= (int)o;
        double zc = z - z0;
        zf[j] = (float)zc;
        wbuf[j] = w;
        mom[0] += w;
        mom[1] = fma(w, w, mom[1]);
        double wz = w * zc;
        mom[2] += wz;
        mom[3] = fma(wz, zc, mom[3]);
        if (P.dbg_z) {
            int jo = P.ev.perm[s0 + j];
            P.dbg_z[jo] = z;
            P.dbg_w[jo] = w * exp(P.ln_shift[ev]);
        }
        A = An;
    }
    block_sum<kEvThreads, 4>(mom, S.red);
    oor = __syncthreads_or(oor);
    if (oor && tid == 0) atomicOr(P.flags + l, CHIM_FLAG_TABLE_RANGE);

    const double sw = mom[0];
    if (!(sw > 0.0)) {   // all-zero event (R15): I = 0
        if (tid == 0) {
            *out = isnan(sw) ? NAN : -INFINITY;
            atomicOr(P.flags + l, CHIM_FLAG_EVENT_ZERO);
            if (P.dbg_h) *P.dbg_h = NAN;
        }
        return;
    }
    double h;
    if (P.bw_rule == CHIM_BW_FIXED) {
        h = P.ev.fixed_bw[ev];
    } else {   // Scott on the weighted sample (R3, O7)
        double s2 = mom[1] / (sw * sw), zb = mom[2] / sw;
        double var = (mom[3] / sw - zb * zb) / (1.0 - s2);
        h = (1.0 - s2 > 0.0 && var > 0.0) ? sqrt(var) * exp(0.2 * log(s2)) : NAN;   // n_eff^(-1/5) = s2^(1/5)
    }
    if (P.dbg_h && tid == 0) *P.dbg_h = h;
    if (!(h > 0.0) || !isfinite(h)) {
        if (tid == 0) {
            *out = NAN;
            atomicOr(P.flags + l, CHIM_FLAG_BW_DEGENERATE);
        }
        if (P.dbg_K) for (int g = tid; g < nz; g += kEvThreads) P.dbg_K[g] = NAN;
        return;
    }

    // ---- scaled coordinates x = z' sqrt(log2(e)/2)/h: exp(-d^2/2h^2) = 2^(-dx^2) --------------------------------
    const double sc = sqrt(kHalfLog2e) / h;
    const float scf = (float)sc;
    const double scd = (double)scf;             // samples and grid are scaled by the SAME rounded factor
    const double wscale = (double)ns / sw;      // weights normalised to mean 1
    const float T = (P.cutoff > 0.0) ? (float)(P.cutoff * sqrt(kHalfLog2e)) : INFINITY;
    const double* zc_g = P.ev.zc + g0;
    const float* qn_g = P.ev.qn + g0;
    const double udz = P.ev.uni_dz[ev];
    const float delta = (float)(udz * scd), xfirst = (float)(zc_g[0] * scd);
    int Bsel = 0;                                // 0 = direct form
    if (udz > 0.0 && T < INFINITY && P.kde_method == CHIM_KDE_AUTO && !P.dbg_K) {
        if (delta * 32.f <= 3.3f) Bsel = 32;
        else if (delta * 16.f <= kMaxBlockSpan) Bsel = 16;
    }
    const int nzp = (int)ev_nz_pad(nz);
    const bool on_grid = P.placement == CHIM_ON_GRID;
    for (int g = tid; g < nzp; g += kEvThreads) {
        float q = 0.f, xg = 0.f;
        if (g < nz) {
            q = qn_g[g];
            if (on_grid)
                q = (float)((double)q * grid_factor(L, P.dc_tab + (size_t)l * (P.n_table + 1 + kZPad), P.n_table + 1 + kZPad,
                                                    P.z_table_max / P.n_table, zc_g[g] + z0));
            xg = (float)(zc_g[g] * scd);
        }
        if (Bsel) {
            const float bd = (float)(g & (Bsel - 1)) * delta;
            q *= ex2_approx(-bd * bd);
            gq[g] = make_float2(q, q);
        } else {
            gq[g] = make_float2(xg, q);
        }
    }
    __syncthreads();

    // ---- S3 + S4: warp passes over 128 consecutive (sorted) samples ----------------------------------------
    const int n_pass = (ns + kPass - 1) / kPass;
    const float inv_delta = (udz > 0.0) ? 1.f / delta : 0.f;
    double lsum = 0.0;                          // this lane's sum_j w_j A_j
    unsigned long long pairs_exec = 0, pairs_cut = 0;
    for (;;) {
        int pass = 0;
        if (lane == 0) pass = atomicAdd(&S.pass_counter, 1);
        pass = __shfl_sync(0xffffffffu, pass, 0);
        if (pass >= n_pass) break;
        const int j0 = pass * kPass + lane * 4;
        const float4 zz = *reinterpret_cast<const float4*>(zf + j0);
        const double2 w01 = *reinterpret_cast<const double2*>(wbuf + j0), w23 = *reinterpret_cast<const double2*>(wbuf + j0 + 2);
        double w[4] = {w01.x, w01.y, w23.x, w23.y};
        float x[4] = {zz.x * scf, zz.y * scf, zz.z * scf, zz.w * scf};
        float xmn = INFINITY, xmx = -INFINITY;
#pragma unroll
        for (int k = 0; k < 4; ++k) {
            const bool valid = (j0 + k < ns) && (w[k] > 0.0);   // zero-weight samples (R15) take no part
            w[k] = valid ? w[k] * wscale : 0.0;
            x[k] = valid ? x[k] : NAN;
            xmn = valid ? fminf(xmn, x[k]) : xmn;
            xmx = valid ? fmaxf(xmx, x[k]) : xmx;
        }
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) {
            xmn = fminf(xmn, __shfl_xor_sync(0xffffffffu, xmn, o));
            xmx = fmaxf(xmx, __shfl_xor_sync(0xffffffffu, xmx, o));
        }
        if (!(xmn <= xmx)) continue;             // no sample of this pass carries weight
#pragma unroll
        for (int k = 0; k < 4; ++k) x[k] = (x[k] == x[k]) ? x[k] : xmn;   // idle slots sit inside the band
        float A[4] = {0.f, 0.f, 0.f, 0.f};
        bool done = false;
        if (Bsel) {
            const float bd = (float)Bsel * delta;
            const int a_lo = max(0, (int)floorf((xmn - T - xfirst) / bd));
            const int a_hi = min(nzp / Bsel - 1, (int)floorf((xmx + T - xfirst) / bd));
            // largest exponent of s^b inside a block: 2 |u| delta (B-1) with |u| <= span + T + B delta
            if (2.f * (xmx - xmn + T + bd) * bd <= kMaxPowExp) {
                if (a_hi >= a_lo) {
                    if (Bsel == 32) power_pass<32>(gq, a_lo, a_hi, xfirst, delta, x, A);
                    else power_pass<16>(gq, a_lo, a_hi, xfirst, delta, x, A);
                    if (lane == 0) pairs_exec += (unsigned long long)(a_hi - a_lo + 1) * Bsel * kPass;
                }
                done = true;
            }
        }
        if (!done) {   // direct form over the band [g_lo, g_hi]
            int g_lo = 0, g_hi = nz - 1;
            if (T < INFINITY) {
                if (udz > 0.0) {
                    g_lo = max(0, (int)floorf((xmn - T - xfirst) * inv_delta));
                    g_hi = min(nz - 1, (int)ceilf((xmx + T - xfirst) * inv_delta));
                } else {
                    const float lo_key = xmn - T, hi_key = xmx + T;
                    int a = 0, b = nz;
                    while (a < b) { int m = (a + b) >> 1; if (gq[m].x < lo_key) a = m + 1; else b = m; }
                    g_lo = a;
                    b = nz;
                    while (a < b) { int m = (a + b) >> 1; if (gq[m].x <= hi_key) a = m + 1; else b = m; }
                    g_hi = a - 1;
                }
            }
            if (Bsel) {   // the q' of this CTA carry the block factor: undo it (rare path: a pass spanning a wide gap)
#pragma unroll 1
                for (int g = g_lo; g <= g_hi; ++g) {
                    const float bdg = (float)(g & (Bsel - 1)) * delta;
                    const float xg = fmaf((float)g, delta, xfirst), q = gq[g].x * ex2_approx(bdg * bdg);
#pragma unroll
                    for (int k = 0; k < 4; ++k) { const float d = xg - x[k]; A[k] = fmaf(q, ex2_approx(-d * d), A[k]); }
                }
            } else if (P.dbg_K) {
#pragma unroll 1
                for (int g = g_lo; g <= g_hi; ++g) {
                    const float2 v = gq[g];
                    float kv = 0.f;
#pragma unroll
                    for (int k = 0; k < 4; ++k) {
                        const float d = v.x - x[k], e = ex2_approx(-d * d);
                        A[k] = fmaf(v.y, e, A[k]);
                        kv = fmaf((float)w[k], e, kv);
                    }
                    double kd = warp_sum((double)kv);
                    if (lane == 0) atomicAdd(P.dbg_K + g, kd);
                }
            } else {
#pragma unroll 2
                for (int g = g_lo; g <= g_hi; ++g) {
                    const float2 v = gq[g];
#pragma unroll
                    for (int k = 0; k < 4; ++k) { const float d = v.x - x[k]; A[k] = fmaf(v.y, ex2_approx(-d * d), A[k]); }
                }
            }
            if (lane == 0 && g_hi >= g_lo) pairs_exec += (unsigned long long)(g_hi - g_lo + 1) * kPass;
        }
#pragma unroll
        for (int k = 0; k < 4; ++k) lsum = fma(w[k], (double)A[k], lsum);
        if (udz > 0.0 && T < INFINITY) {   // algorithmic pair count: grid points within the cut-off of each weighted sample
#pragma unroll
            for (int k = 0; k < 4; ++k)
                if (w[k] > 0.0) {
                    const int a = max(0, (int)ceilf((x[k] - T - xfirst) * inv_delta)), b = min(nz - 1, (int)floorf((x[k] + T - xfirst) * inv_delta));
                    pairs_cut += (unsigned long long)max(0, b - a + 1);
                }
        } else if (lane == 0) {
            pairs_cut += (unsigned long long)nz * min(kPass, ns - pass * kPass);
        }
    }
    // K(z) = 1/(N_s h sqrt(2 pi)) sum_j w_j exp(..): undo the weight normalisation (sw/ns)
    const double knorm = (sw / ns) / ((double)ns * h * 2.50662827463100050242);
    double tot[3] = {lsum, (double)pairs_exec, (double)pairs_cut};
    block_sum<kEvThreads, 3>(tot, S.red);
    if (tid == 0 && P.stats) {
        if (tot[1] > 0.0) atomicAdd(P.stats, (unsigned long long)tot[1]);
        if (tot[2] > 0.0) atomicAdd(P.stats + 1, (unsigned long long)tot[2]);
    }
    if (P.dbg_K) {   // diagnostics: turn the accumulated sums into K(z_g)
        __syncthreads();
        const double ks = knorm * exp(P.ln_shift[ev]);
        for (int g = tid; g < nz; g += kEvThreads) P.dbg_K[g] *= ks;
    }
    if (tid == 0) {
        double I = tot[0] * knorm;
        if (I > 0.0) *out = log(I) + P.ln_shift[ev] + P.ln_qscale[ev];
        else if (I == 0.0) { *out = -INFINITY; atomicOr(P.flags + l, CHIM_FLAG_EVENT_ZERO); }
        else *out = NAN;
    }
}

size_t events_smem_bytes(int max_ns, int max_nz) {
    return ((sizeof(EvSmem) + 15) / 16) * 16 + (sizeof(double) + sizeof(float)) * ev_ns_pad((size_t)max_ns) +
           ev_aux_bytes((size_t)max_nz);
}

cudaError_t launch_events(const EventKernelParams& P, cudaStream_t st) {
    size_t smem = events_smem_bytes(P.ev.max_ns, P.ev.max_nz);
    cudaError_t e = cudaFuncSetAttribute(k_events, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    if (e != cudaSuccess) return e;
    long long nb = (P.dbg_event >= 0) ? P.n_lambda : (long long)P.n_lambda * P.ev.n_events;
    if (nb <= 0) return cudaSuccess;
    k_events<<<(unsigned)nb, kEvThreads, smem, st>>>(P);
    return cudaGetLastError();
}

}  // namespace chim
