// k_events.cu -- steps S2 + S3 + S4 fused: one CTA per (event, lambda).
//
//   S2  per posterior sample: z_j, source masses, log2 of the population weight, all fp32.
//       Narrow events (samples spanning <= 0.9 in ln d_L; every BASELINE config): event-local polynomials in ln d_L fitted
//       per (event, lambda) by k_polyfit (poly_sample, chim_internal.cuh); 24-byte records streamed from L2 with
//       coalesced 128 + 64-bit loads, the event's slice of the per-lambda mass table staged by a TMA bulk copy.
//       Wide events: the per-lambda z(ln d_L) table rows (sample_eval; rows staged by TMA when they fit, hi + lo pairs
//       where differences cancel).  A second sweep over shared memory turns log2 w into w / max w and forms the weighted
//       moments -> Scott bandwidth h (R3).  z_j and w_j never leave shared memory.
//   S3+S4  I_i = sum_g q_g K(z_g) = (1/(N_s h sqrt(2 pi))) sum_j w_j A_j,  A_j = sum_g q_g exp(-(z_g - z_j)^2 / 2h^2),
//       q_g = p_gal(z_g) x trapezoid weight (eq. 19 evaluated on the grid, eq. 14).
//       Three formulations:
//
//       local-expansion form (equally spaced grid; the default): A(y) is expanded about box centres
//       placed on grid points -- Hermite generating function, 12 terms, one coefficient table per CTA -- and every
//       sample costs one degree-11 polynomial (packed FFMA2) instead of ~2 t h / dz Gaussian pairs (le_phase).
//
//       power form (equally spaced grid; when the expansion does not fit): with x = z sqrt(log2(e)/2)/h, delta the
//       grid spacing in x, block start x_a, u = x_a - x_j and g = aB + b:
//           2^-(x_g - x_j)^2 = 2^(-u^2) * (2^(-2 delta u))^b * 2^(-b^2 delta^2)
//       so per block of B grid points  sum_b q_g E_gj = e0 * sum_b q'_b s^b  with q'_b = q_g 2^(-b^2 delta^2)
//       precomputed per CTA: a Horner polynomial in s -- ONE fp32 FMA per pair, issued as packed FFMA2 (two
//       samples per instruction), and two MUFU.EX2 (e0, s) per sample and block.  Samples in lanes (4 per lane, 128 per
//       warp pass, sorted in z); a pass visits the grid band within t*h of its samples (R9).
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
#ifndef CHIM_S2_UNROLL
#define CHIM_S2_UNROLL 2
#endif
constexpr int kS2Unroll = CHIM_S2_UNROLL;
constexpr int kEvThreads = CHIM_EV_THREADS;   // 256 x 3 CTAs per SM measured faster than 384 x 2 and 512 x 1
constexpr int kPass = 128;               // samples per warp pass (4 per lane)
constexpr float kMaxBlockSpan = 4.8f;    // B * delta limit of the power form
constexpr float kMaxPowExp = 100.f;      // bound on log2 of the largest s^b inside a block (fp32 overflow guard)
constexpr int kRowStage = 224;           // rows of the z(ln d_L) table staged per CTA (14 KB)
constexpr int kMassStage = 384;          // mass-table rows staged per CTA and variant (2 x 6 KB)

constexpr int kLeP = 12;                 // terms of the local expansion (degree 11)
constexpr int kLeMaxBox = 96;            // boxes per event the local-expansion form accepts
constexpr float kLeMaxW = 1.3f;          // largest box width in units of sqrt(2) h (truncation error)

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
    unsigned long long kred[kEvThreads / 32];
    double mom[4], slev;      // W, Q, B, A of Scott's rule about the heaviest sample (relative to level slev, R21)
    int careful;
    unsigned long long mbar;
    int pass_counter;
    int mass_lo, mass_fit, early_tma;
    double h, scd;            // bandwidth and the coordinate scale (as the rounded float, widened)
    float scf, delta, xfirst; // scale, grid spacing and first grid point in scaled coordinates
    int Bsel;                 // block size of the power form, 0 = direct form
    // local-expansion form (le_nbox > 0): coordinates y = z'/(sqrt(2) h)
    float scy, dy, yfirst;    // scale, grid spacing and first grid point in y
    int le_m, le_D, le_blo, le_nbox;   // grid points per box, half-width of the psi table, first box, number of boxes
    // event-local polynomials of S2 (use_poly != 0): z - z0 [7], ln(1+z) [7], 1/(1+z) [7], smooth log2 factor [7]
    alignas(16) float poly[4 * kPolyN];
    // lambda-independent scalars of the event, fetched once beside the constants (one L2 latency instead of one per use)
    double ev_udz, ev_zfirst, ev_ln_out;   // grid spacing (0: not equally spaced), first centred grid point, ln_shift + ln_qscale
    double ev_maxdz;          // largest grid spacing of the event
    int exact;                // S3 in log space without cut-off (exact_log2_kde)
};

__host__ __device__ inline size_t ev_ns_pad(size_t ns) { return (ns + kPass - 1) / kPass * kPass; }
__host__ __device__ inline size_t ev_nz_pad(size_t nz) { return (nz + 31) / 32 * 32; }
__host__ __device__ inline size_t ev_aux_bytes(size_t nz) {   // S2: staged table + mass rows; S3: (q', q') or (x_g, q_g) per grid point
    size_t a = sizeof(float2) * ev_nz_pad(nz), b = (size_t)kRowStage * sizeof(Row) + 2 * (size_t)kMassStage * sizeof(MassRow);
    return a > b ? a : b;
}

// One block of B grid points for the 4 samples of a lane: tot_k += 2^(-u_k^2) * sum_b q'_b s_k^b (Horner, FFMA2).
template <int B>
__device__ __forceinline__ void power_block(const float4* __restrict__ qp, f32x2 xs2, f32x2 cs2, f32x2 nx01, f32x2 nx23,
                                            f32x2& tot01, f32x2& tot23) {
    const f32x2 u01 = add2(xs2, nx01), u23 = add2(xs2, nx23);          // u = x_a - x_j
    const f32x2 su01 = mul2(u01, cs2), su23 = mul2(u23, cs2);          // -2 delta u
    const f32x2 q01 = mul2(u01, u01), q23 = mul2(u23, u23);            // u^2
    float a, b, c, d;
    unpack2(su01, a, b);
    unpack2(su23, c, d);
    const f32x2 s01 = pack2(ex2f(a), ex2f(b)), s23 = pack2(ex2f(c), ex2f(d));
    unpack2(q01, a, b);
    unpack2(q23, c, d);
    const f32x2 e01 = pack2(ex2f(-a), ex2f(-b)), e23 = pack2(ex2f(-c), ex2f(-d));
    f32x2 a01 = 0ull, a23 = 0ull;     // (+0.f, +0.f)
#pragma unroll
    for (int i = B / 4 - 1; i >= 0; --i) {
        const float4 v = qp[i];       // q'_4i .. q'_4i+3: one shared-memory wavefront pair feeds 8 packed FMAs
        const f32x2 q3 = pack2(v.w, v.w), q2 = pack2(v.z, v.z), q1 = pack2(v.y, v.y), q0 = pack2(v.x, v.x);   // (scalar operand of FFMA2)
        a01 = fma2(a01, s01, q3);
        a23 = fma2(a23, s23, q3);
        a01 = fma2(a01, s01, q2);
        a23 = fma2(a23, s23, q2);
        a01 = fma2(a01, s01, q1);
        a23 = fma2(a23, s23, q1);
        a01 = fma2(a01, s01, q0);
        a23 = fma2(a23, s23, q0);
    }
    tot01 = fma2(e01, a01, tot01);
    tot23 = fma2(e23, a23, tot23);
}

template <int B>
__device__ __forceinline__ void power_pass(const float* __restrict__ gq, int a_lo, int a_hi, float xfirst, float delta,
                                           const float (&x)[4], float (&A)[4]) {
    f32x2 tot01 = 0ull, tot23 = 0ull;
    const float cs = -2.f * delta, bd = (float)B * delta;
    const f32x2 cs2 = pack2(cs, cs), nx01 = pack2(-x[0], -x[1]), nx23 = pack2(-x[2], -x[3]);
    float af = (float)a_lo;
    const float4* qp = reinterpret_cast<const float4*>(gq + a_lo * B);
#pragma unroll 1
    for (int a = a_lo; a <= a_hi; ++a) {
        const float xs = fmaf(af, bd, xfirst);     // exact block origin: no drift from block to block
        power_block<B>(qp, pack2(xs, xs), cs2, nx01, nx23, tot01, tot23);
        af += 1.0f;
        qp += B / 4;
    }
    unpack2(tot01, A[0], A[1]);
    unpack2(tot23, A[2], A[3]);
}

// ---- local-expansion form of S3 + S4 (equally spaced grid) -------------------------------------------------
// With y = z'/(sqrt(2) h):  I ~ sum_j w_j A(y_j),  A(y) = sum_g q_g exp(-(y_g - y)^2).  In units of h the samples are far
// denser than the grid, and A is entire, so A is expanded about box centres c_b placed on grid points (box = m grid
// spacings ~ one unit of y):  exp(-(t - s)^2) = sum_n psi_n(t) s^n,  psi_n(t) = exp(-t^2) H_n(t)/n!  (generating function of
// the Hermite polynomials), t = y_g - c_b, s = y - c_b, |s| <= w/2:
//     A(y) = sum_{n<P} B_bn s^n + O((w/sqrt 2)^P / sqrt(P!)),   B_bn = sum_{|d| <= D} q_{g_b+d} psi_n(d dy)
// (grid points beyond the cut-off t*h of the box are dropped: R9).  Because the centres sit on grid points, psi_n(d dy)
// is ONE table per CTA, shared by all boxes (psi_n(-t) = (-1)^n psi_n(t)).  Per sample: one degree-(P-1) Horner
// polynomial (packed FFMA2) instead of ~2 t h / dz Gaussian pairs.  P = 12, w <= 1.3: truncation < 1e-8 of A.
struct LeSmem {
    float* qs;      // [nzp]  q_g (x grid factor for placement ON_GRID), 0 beyond the grid
    float* psi;     // [(D+1) * kLeP]
    float* Bc;      // [nbox * kLeP]
};
__host__ __device__ inline size_t le_bytes(size_t nzp, int D, int nbox) {
    return 4 * nzp + 4 * (size_t)kLeP * (D + 1) + 4 * (size_t)kLeP * nbox + 64;
}
__device__ __forceinline__ LeSmem le_layout(unsigned char* aux, size_t nzp, int D, int nbox) {
    LeSmem M;
    M.qs = reinterpret_cast<float*>(aux);
    M.psi = M.qs + nzp;
    M.Bc = M.psi + (size_t)kLeP * (D + 1);
    return M;
}

// psi table of the local-expansion form: thread d computes psi_0..psi_{P-1} at t = d dy by the three-term recurrence
// (threads from the top of the CTA, so that the warps staging q_g and the warps building psi overlap)
__device__ __forceinline__ void le_psi_table(float* __restrict__ psi, int D, float dy) {
    for (int d = kEvThreads - 1 - (int)threadIdx.x; d <= D; d += kEvThreads) {
        const float t = (float)d * dy, t2 = 2.f * t;
        float p0 = ex2f(-t * t * 1.44269504088896341f), p1 = t2 * p0;
        float* o = psi + (size_t)d * kLeP;
        o[0] = p0;
        o[1] = p1;
#pragma unroll
        for (int n = 1; n < kLeP - 1; ++n) {
            const float p2 = fmaf(t2, p1, -2.f * p0) * (1.0f / (float)(n + 1));
            o[n + 1] = p2;
            p0 = p1;
            p1 = p2;
        }
    }
}

// Called by all threads after qs and psi have been staged (and a barrier).  Returns this lane's sum_j w_j A_j.
template <bool kStats>
__device__ double le_phase(const EvSmem& S, const LeSmem& M, const float* __restrict__ zf, const float* __restrict__ wl,
                           int ns, int nz, float Ty, unsigned long long& fma_ops, unsigned long long& pairs_cut) {
    const int tid = threadIdx.x, lane = tid & 31, wid = tid >> 5;
    const float scy = S.scy, dy = S.dy, yfirst = S.yfirst;
    const int m = S.le_m, D = S.le_D, b_lo = S.le_blo, nbox = S.le_nbox;
    const float wbox = (float)m * dy;
    // (b) coefficients: item = (box, quad of n, quarter of the d range); the four quarters sit in adjacent lanes
    const int H = D >> 1, n_items = nbox * 12;
    for (int base = 0; base < n_items; base += kEvThreads) {
        const int id = base + tid;
        const bool valid = id < n_items;
        const int i = valid ? id / 12 : 0, rem = id - (id / 12) * 12, quad = rem >> 2, seg = rem & 3;
        const int gc = (b_lo + i) * m;
        const bool neg = seg < 2;
        int d0 = (seg == 0 || seg == 3) ? H + 1 : (seg == 1 ? 1 : 0), d1 = (seg == 0 || seg == 3) ? D : H;
        // clip to the grid: g = gc -/+ d in [0, nz)
        if (neg) { d0 = max(d0, gc - (nz - 1)); d1 = min(d1, gc); }
        else { d0 = max(d0, -gc); d1 = min(d1, nz - 1 - gc); }
        if (!valid) d1 = d0 - 1;
        f32x2 axy = 0ull, azw = 0ull;      // (+0.f, +0.f): accumulators of n = 4 quad + {0, 1} and + {2, 3}, packed for FFMA2
        const float* qp = M.qs + gc + (neg ? -d0 : d0);
        const int qstep = neg ? -1 : 1;
        const ulonglong2* pp = reinterpret_cast<const ulonglong2*>(M.psi) + quad + d0 * (kLeP / 4);
        int n = d1 - d0 + 1;
#pragma unroll 1
        for (; n >= 4; n -= 4) {
#pragma unroll
            for (int k = 0; k < 4; ++k) {
                const float q = qp[k * qstep];
                const ulonglong2 v = pp[k * (kLeP / 4)];
                const f32x2 q2 = pack2(q, q);
                axy = fma2(q2, v.x, axy);
                azw = fma2(q2, v.y, azw);
            }
            qp += 4 * qstep;
            pp += 4 * (kLeP / 4);
        }
        for (; n > 0; --n) {
            const float q = *qp;
            const ulonglong2 v = *pp;
            const f32x2 q2 = pack2(q, q);
            axy = fma2(q2, v.x, axy);
            azw = fma2(q2, v.y, azw);
            qp += qstep;
            pp += kLeP / 4;
        }
        float4 acc;
        unpack2(axy, acc.x, acc.y);
        unpack2(azw, acc.z, acc.w);
        if (neg) { acc.y = -acc.y; acc.w = -acc.w; }   // psi_n(-t) = (-1)^n psi_n(t); n = 4 quad + {0,1,2,3}
#pragma unroll
        for (int o = 1; o <= 2; o <<= 1) {
            acc.x += __shfl_xor_sync(0xffffffffu, acc.x, o);
            acc.y += __shfl_xor_sync(0xffffffffu, acc.y, o);
            acc.z += __shfl_xor_sync(0xffffffffu, acc.z, o);
            acc.w += __shfl_xor_sync(0xffffffffu, acc.w, o);
        }
        if (valid && seg == 0) reinterpret_cast<float4*>(M.Bc)[i * (kLeP / 4) + quad] = acc;
        if (kStats && valid) fma_ops += 4ull * (unsigned long long)max(0, d1 - d0 + 1);
    }
    __syncthreads();
    // (c) evaluation: a warp pass = 128 consecutive (sorted) samples, 4 per lane; the boxes the pass touches are visited in
    //     turn (usually one or two), each lane keeping the value of the box its sample lies in
    const float inv_w = 1.0f / wbox, inv_dy = 1.0f / dy;
    const int n_pass = (ns + kPass - 1) / kPass;
    double lsum = 0.0;
    for (int pass = wid; pass < n_pass; pass += kEvThreads / 32) {
        const int j0 = pass * kPass + lane * 4;
        const float4 zz = *reinterpret_cast<const float4*>(zf + j0);     // padded: idle slots repeat the last sample, w = 0
        const float4 ww = *reinterpret_cast<const float4*>(wl + j0);
        const float y[4] = {zz.x * scy, zz.y * scy, zz.z * scy, zz.w * scy};
        int bx[4];
#pragma unroll
        for (int r = 0; r < 4; ++r) bx[r] = min(max((int)floorf(fmaf(y[r] - yfirst, inv_w, 0.5f)) - b_lo, 0), nbox - 1);
        // the samples are sorted (up to fp32 rounding, which at worst moves a sample to the neighbouring box, where the
        // expansion is still valid): the pass spans the boxes of its first and last sample
        const int bmin = __shfl_sync(0xffffffffu, bx[0], 0), bmax = __shfl_sync(0xffffffffu, bx[3], 31);
        bx[0] = min(max(bx[0], bmin), bmax);
        bx[3] = min(max(bx[3], bx[0]), bmax);
        bx[1] = min(max(bx[1], bx[0]), bx[3]);
        bx[2] = min(max(bx[2], bx[0]), bx[3]);
        float A[4] = {0.f, 0.f, 0.f, 0.f};
        for (int i = bmin; i <= bmax; ++i) {
            const bool mine = (bx[0] <= i) & (bx[3] >= i);               // sorted within the lane as well
            if (!__any_sync(0xffffffffu, mine)) continue;                 // empty box inside the pass
            const float c = fmaf((float)((b_lo + i) * m), dy, yfirst);
            const float4* bp = reinterpret_cast<const float4*>(M.Bc) + i * (kLeP / 4);
            const float4 c0 = bp[0], c1 = bp[1], c2 = bp[2];
            const f32x2 s01 = pack2(y[0] - c, y[1] - c), s23 = pack2(y[2] - c, y[3] - c);
            f32x2 a01 = pack2(c2.w, c2.w), a23 = a01;
#define CHIM_LE_STEP(cf) { const f32x2 q_ = pack2(cf, cf); a01 = fma2(a01, s01, q_); a23 = fma2(a23, s23, q_); }
            CHIM_LE_STEP(c2.z) CHIM_LE_STEP(c2.y) CHIM_LE_STEP(c2.x)
            CHIM_LE_STEP(c1.w) CHIM_LE_STEP(c1.z) CHIM_LE_STEP(c1.y) CHIM_LE_STEP(c1.x)
            CHIM_LE_STEP(c0.w) CHIM_LE_STEP(c0.z) CHIM_LE_STEP(c0.y) CHIM_LE_STEP(c0.x)
#undef CHIM_LE_STEP
            float v[4];
            unpack2(a01, v[0], v[1]);
            unpack2(a23, v[2], v[3]);
#pragma unroll
            for (int r = 0; r < 4; ++r) A[r] = (bx[r] == i) ? v[r] : A[r];
        }
        lsum += (double)fmaf(ww.x, A[0], fmaf(ww.y, A[1], fmaf(ww.z, A[2], ww.w * A[3])));
        if (kStats) {
            const float wv[4] = {ww.x, ww.y, ww.z, ww.w};
#pragma unroll
            for (int r = 0; r < 4; ++r)
                if (wv[r] > 0.f) {
                    const int a = max(0, (int)ceilf((y[r] - Ty - yfirst) * inv_dy)), b = min(nz - 1, (int)floorf((y[r] + Ty - yfirst) * inv_dy));
                    pairs_cut += (unsigned long long)max(0, b - a + 1);
                    fma_ops += kLeP;
                }
        }
    }
    return lsum;
}

// S2 sweep 1 over the event's samples: z_j - z0 and log2 w_j to shared memory; returns the thread's max log2 w and (jx) the
// first sample that attains it.
template <bool kStaged>
__device__ __forceinline__ float s2_sweep(const float4* __restrict__ rec, const LamF& Fs, const float4* __restrict__ rows,
                                          int k_base, const MassLookup& M, int ns, float z0h, float z0l,
                                          float* __restrict__ zf, float* __restrict__ wl, int& jx) {
    float mx = -INFINITY;
    jx = 0;
    const int tid = threadIdx.x;
    const LamF F = Fs;                               // registers, not re-read from shared memory after every store
    const int ns32 = (ns + 31) & ~31;                // whole warps stay in the loop (sample_eval votes)
    Rec R = ldg_stream_rec(rec + 2 * min(tid, ns - 1));
#pragma unroll(kS2Unroll)
    for (int j = tid; j < ns32; j += kEvThreads) {
        const float4 A = R.A, Bq = R.B;
        if (j + kEvThreads < ns32) R = ldg_stream_rec(rec + 2 * min(j + kEvThreads, ns - 1));   // one iteration ahead
        const uint32_t tkq = __float_as_uint(A.x);
        const int k = (int)(tkq >> kTkFracBits);     // in [1, K]: clamped when the records were packed
        const float t = __uint_as_float(0x3F800000u | ((tkq << (32 - kTkFracBits)) >> 9)) - 1.0f;
        const bool in_range = tkq <= F.tkmax_ev_q;
        float4 q0, q1, q2, q3;
        if (kStaged) {
            const float4* r = rows + 4 * (k - k_base);
            q0 = r[0]; q1 = r[1]; q2 = r[2]; q3 = r[3];
        } else {
            const float4* r = rows + 4 * (size_t)k;
            q0 = __ldg(r); q1 = __ldg(r + 1); q2 = __ldg(r + 2); q3 = __ldg(r + 3);
        }
        float zc, l2w;
        sample_eval(F, q0, q1, q2, q3, t, z0h, z0l, A.y, A.z, A.w, Bq.x, Bq.y, Bq.z, Bq.w, M, in_range, zc, l2w);
        if (j < ns) {
            zf[j] = zc;
            wl[j] = l2w;
            if (l2w > mx) { mx = l2w; jx = j; }
        }
    }
    return mx;
}

// S2 sweep 1 with the event-local polynomials (poly_sample, chim_internal.cuh): z_j - z0 and log2 w_j to shared memory.
// kFit: every mass-table row the event can address is staged (the tm clamp keeps the index inside the stage).
// All samples of an event on this path lie inside the table (use_poly), so there is no range check.
template <bool kFit>
__device__ __forceinline__ float s2_sweep_poly(const float4* __restrict__ pa, const float2* __restrict__ pb, const LamF& Fs,
                                               const float* __restrict__ pc, const MassLookup& M, int ns,
                                               float* __restrict__ zf, float* __restrict__ wl, int& jx) {
    float mx = -INFINITY;
    jx = 0;
    const int tid = threadIdx.x;
    const LamF F = Fs;
    PolyCoef C;
    load_poly(C, pc);
    const int ns32 = (ns + 31) & ~31;                // the records are padded to ns32 with copies of the last sample
    // clamp of the mass-table coordinate: the table's range, and (kFit) the staged rows [M.lo, M.lo + M.cap)
    const float tm_lo = kFit ? fmaxf(1.0f, (float)M.lo) : 1.0f;
    const float tm_hi = kFit ? fminf(F.tm_max, (float)(M.lo + M.cap) - 0.01f) : F.tm_max;
    pa += tid;
    pb += tid;
    PRec R = ldg_stream_prec(pa, pb);                // unconditional: the record arrays carry a tail of 2 x 256 spare records
#pragma unroll 2
    for (int j = tid; j < ns32; j += kEvThreads) {
        const float4 A = R.A;
        const float2 Bq = R.B;
        pa += kEvThreads;
        pb += kEvThreads;
        R = ldg_stream_prec(pa, pb);                 // one iteration ahead (past the event: read and dropped)
        float zc, l2w;
        poly_sample<kFit>(F, F.gk2, F.cpsi, C, A, Bq, M, tm_lo, tm_hi, zc, l2w);
        if (j < ns) {
            zf[j] = zc;
            wl[j] = l2w;
            if (l2w > mx) { mx = l2w; jx = j; }
        }
    }
    return mx;
}

// Block-wide argmax of (value, first index): every thread passes its own candidate; the result is valid in all threads.
// Key = order-preserving bits of the float in the upper word, ~index in the lower one (ties: the smallest index wins).
// A NaN value sorts above everything (it is reported by the caller).  Two barriers; kscratch holds kEvThreads/32 keys.
__device__ __forceinline__ void block_argmax(float& v, int& j, unsigned long long* kscratch) {
    const uint32_t b = __float_as_uint(v);
    unsigned long long key = ((unsigned long long)(b ^ ((b >> 31) ? 0xFFFFFFFFu : 0x80000000u)) << 32) | (uint32_t)(~(uint32_t)j);
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) {
        const unsigned long long other = __shfl_xor_sync(0xffffffffu, key, o);
        key = other > key ? other : key;
    }
    __syncthreads();                              // protect kscratch from a previous use
    if ((threadIdx.x & 31) == 0) kscratch[threadIdx.x >> 5] = key;
    __syncthreads();
#pragma unroll
    for (int k = 0; k < kEvThreads / 32; ++k) { const unsigned long long other = kscratch[k]; key = other > key ? other : key; }
    const uint32_t hb = (uint32_t)(key >> 32);
    v = __uint_as_float(hb ^ ((hb >> 31) ? 0x80000000u : 0xFFFFFFFFu));
    j = (int)(~(uint32_t)key);
}

// S3 + S4 without cut-off and in log space, for the units the fp32 pair loop cannot represent (R9, R21): an event left with a
// few samples within ~1e-4 of each other has a bandwidth far below the grid spacing, so that no grid point lies within t h
// of any sample and the nearest ones contribute e^-100 -- small, not zero.  Returns log2 of
//     sum_j w_j sum_g q_g exp(-(z_g - z_j)^2 / 2h^2)
// (block-uniform; -inf if every term is zero) by two passes over all (weighted sample, grid point) pairs: the largest
// exponent, then the sum relative to it.  Slow by design: only taken when t h < half a grid spacing or the fast sum is 0.
__device__ __noinline__ double exact_log2_kde(const LamConst& L, const double* __restrict__ dc_row, int dc_nodes, double dc_dz,
                                              const float* __restrict__ zf, const float* __restrict__ wl, int ns3,
                                              const double* __restrict__ zc_g, const float* __restrict__ qn_g, int nz, double z0,
                                              double h, double* red, unsigned long long* kred) {
    const int tid = threadIdx.x;
    const double sc = sqrt(kHalfLog2e) / h;
    const bool on_grid = dc_row != nullptr;     // placement ON_GRID: psi/J on the grid points
    float mxt = -INFINITY;
    int dummy = 0;
    double sum = 0.0;
    float M = 0.f;
#pragma unroll 1
    for (int pass = 0; pass < 2; ++pass) {
        for (int g = tid; g < nz; g += kEvThreads) {
            double q = (double)qn_g[g];
            if (on_grid && q > 0.0) q *= grid_factor(L, dc_row, dc_nodes, dc_dz, zc_g[g] + z0);
            if (!(q > 0.0)) continue;
            const float lq = (float)log2(q);
            const double xg = zc_g[g] * sc;
            for (int j = 0; j < ns3; ++j) {
                const float w = wl[j];
                if (!(w > 0.f)) continue;
                const double d = xg - (double)zf[j] * sc;
                const float term = lg2f(w) + lq - (float)(d * d);
                if (pass == 0) mxt = fmaxf(mxt, term);
                else sum += (double)ex2f(term - M);
            }
        }
        if (pass == 0) {
            block_argmax(mxt, dummy, kred);
            M = mxt;
            if (!(M > -INFINITY)) return -INFINITY;
        }
    }
    double t1[1] = {sum};
    block_sum<kEvThreads, 1>(t1, red);
    return (double)M + log2(t1[0]);
}

// shared-memory layout after EvSmem: zf float[ns_pad] | wl float[ns_pad] | aux = staged table rows + mass rows (S2) / gq float2[nz_pad] (S3)
// One (event, lambda) unit.  Block-uniform returns only.  again: the CTA has processed a unit before (work-list mode): the
// one-shot mbarrier is invalidated and initialised anew.
template <bool kStats>
__device__ __forceinline__ void events_unit(const EventKernelParams& P, const int l, const int ev, unsigned char* smem_raw, const bool again,
                                            const bool force_careful) {
    EvSmem& S = *reinterpret_cast<EvSmem*>(smem_raw);
    float* zf = reinterpret_cast<float*>(smem_raw + ((sizeof(EvSmem) + 127) / 128) * 128);
    const size_t ns_pad = ev_ns_pad(P.ev.max_ns);
    float* wl = zf + ns_pad;
    unsigned char* aux = reinterpret_cast<unsigned char*>(wl + ns_pad);
    float2* gq = reinterpret_cast<float2*>(aux);     // direct form: (x_g, q_g)
    float* gqp = reinterpret_cast<float*>(aux);      // power form: q'_g
    float4* rows_s = reinterpret_cast<float4*>(aux);
    MassRow* mass_s = reinterpret_cast<MassRow*>(aux + (size_t)kRowStage * sizeof(Row));
    const int tid = threadIdx.x, lane = tid & 31, wid = tid >> 5;

    const int64_t s0 = P.ev.sample_off[ev], g0 = P.ev.grid_off[ev];
    const int ns = (int)(P.ev.sample_off[ev + 1] - s0), nz = (int)(P.ev.grid_off[ev + 1] - g0);
    double* out = (P.dbg_event >= 0) ? P.logI + l : P.logI + (size_t)l * P.ev.n_events + ev;
    const Row* tab = P.tab + (size_t)l * P.tab_rows;
    const MassRow* mtab = P.mtab + (size_t)l * 2 * (P.n_mass + 2);
    const int k_lo = P.ev.k_lo[ev], k_hi = P.ev.k_hi[ev];       // table rows the event's samples address
    const bool staged = (k_hi - k_lo + 1) <= kRowStage;
    const int mcap = min(kMassStage, P.n_mass + 2);

    {   // stage the per-lambda constants in shared memory
        const int nw = sizeof(LamConst) / 4;
        const uint32_t* src = reinterpret_cast<const uint32_t*>(P.Lc + l);
        uint32_t* dst = reinterpret_cast<uint32_t*>(&S.L);
        for (int i = tid; i < nw; i += kEvThreads) dst[i] = src[i];
        if (tid == 0) {
            S.pass_counter = 0;
            if (again) {
                // work-list mode: the previous unit of this CTA wrote the staged regions (grid factors, psi coefficients, rows)
                // with ordinary stores; the bulk copies below write the same shared memory through the async proxy.  The
                // __syncthreads after the previous unit ordered those stores before this point for the generic proxy only:
                // the cross-proxy fence makes them visible to (ordered before) the async-proxy writes that follow.
                asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
                asm volatile("mbarrier.inval.shared::cta.b64 [%0];" ::"r"(smem_u32(&S.mbar)) : "memory");
            }
            mbar_init(&S.mbar, 1);
            // polynomial path: the stage bounds were computed by k_polyfit, so the TMA copy of the mass rows starts now and
            // runs beside the staging of the constants (the same test as use_poly below, on the global copy of the constants)
            const double h0 = P.ev.tk_h[ev], c0 = P.ev.tk_c[ev];
            const float* pr = P.poly + ((size_t)l * P.ev.n_events + ev) * (4 * kPolyN);
            int early = 0;
            if (h0 > 0.0 && P.Lc[l].flags == 0 && c0 + h0 < P.Lc[l].tkmax_ev) {
                const int mlo = __float_as_int(__ldg(pr + 26)), nr = __float_as_int(__ldg(pr + 27));
                const uint32_t mbytes = (uint32_t)abs(nr) * (uint32_t)sizeof(MassRow);
                S.mass_lo = mlo;
                S.mass_fit = nr > 0 ? 1 : 0;
                mbar_expect_tx(&S.mbar, 2 * mbytes);
                bulk_g2s(mass_s, mtab + mlo, mbytes, &S.mbar);
                bulk_g2s(mass_s + mcap, mtab + (P.n_mass + 2) + mlo, mbytes, &S.mbar);
                early = 1;
            }
            S.early_tma = early;
        }
        if (tid == 32) {
            const double a = P.ev.uni_dz[ev], b = P.ev.zc[g0], c = P.ln_shift[ev], d = P.ln_qscale[ev], e = P.ev.max_dz[ev];
            S.ev_udz = a; S.ev_zfirst = b; S.ev_ln_out = c + d; S.ev_maxdz = e;
        }
    }
    __syncthreads();
    const LamConst& L = S.L;
    if (L.flags) {   // invalid lambda: NaN
        if (tid == 0) *out = NAN;
        return;
    }
    const double z0 = P.ev.z0[ev];
    // event-local polynomials (S2): narrow d_L range and every node inside the table
    const double tk_h = P.ev.tk_h[ev], tk_c = P.ev.tk_c[ev];
    const bool use_poly = tk_h > 0.0 && tk_c + tk_h < L.tkmax_ev;
    if (use_poly && tid < 4 * kPolyN) S.poly[tid] = P.poly[((size_t)l * P.ev.n_events + ev) * (4 * kPolyN) + tid];   // fitted by k_polyfit

    // ---- TMA: the event's slice of the z(ln d_L) table and the mass-table rows it can address: ln m1 = ln m1d - ln(1+z),
    //      z between the event's first and last (sorted) sample; rows outside the staged range fall back to global
    //      memory inside sample_eval ----------------------------------------------------------------------------
    if (tid == 0 && !S.early_tma) {
        const float u_lo = tab[k_lo].u0, u_hi = tab[min(k_hi + 1, P.tab_rows - 1)].u0;   // ln(1+z) at the bracketing nodes
        const int ma = max(1, min((int)fma(P.ev.lnm1_lo[ev] - (double)u_hi - L.lm0, L.inv_dlm, 1.0), P.n_mass));
        const int mb = max(1, min((int)fma(P.ev.lnm1_hi[ev] - (double)u_lo - L.lm0, L.inv_dlm, 1.0), P.n_mass));
        int mlo = ma - 1 + max(0, (mb - ma + 3 - mcap) / 2);                              // wider than the stage: keep the centre
        mlo = max(0, min(mlo, P.n_mass + 2 - mcap));
        S.mass_lo = mlo;
        S.mass_fit = (mb - ma + 3 <= mcap) ? 1 : 0;
        const uint32_t rb = (staged && !use_poly) ? (uint32_t)(k_hi - k_lo + 1) * (uint32_t)sizeof(Row) : 0u, mbytes = (uint32_t)min(mcap, mb + 3 - mlo) * (uint32_t)sizeof(MassRow);   // rows mlo .. mb + 2: what the event can address (+ margin), not the whole stage
        mbar_expect_tx(&S.mbar, rb + 2 * mbytes);
        if (rb) bulk_g2s(rows_s, tab + k_lo, rb, &S.mbar);
        bulk_g2s(mass_s, mtab + mlo, mbytes, &S.mbar);
        bulk_g2s(mass_s + mcap, mtab + (P.n_mass + 2) + mlo, mbytes, &S.mbar);
    }
    __syncthreads();     // publishes S.mass_lo
    MassLookup M;
    M.g = mtab;
    M.s = mass_s;
    M.lo = S.mass_lo;
    M.cap = mcap;
    M.n_mass = P.n_mass;
    mbar_wait(&S.mbar, 0);

    // ---- S2: z_j - z0 and the weights, relative to the heaviest sample d; moments for Scott's rule --------------------
    // Scott's rule (R3, R21) is evaluated about and excluding d: with w_d = 1, u = z - z_d and, over j != d,
    // W = sum w, Q = sum w^2, B = sum w u, A = sum w u^2:  var = [A(1+W) - B^2]/[2W + W^2 - Q], n_eff = (1+W)^2/(1+Q) -- no
    // cancellation however few samples carry the event.  The fast sweep (fp32 polynomials) is redone by the careful one
    // (table rows with hi + lo pairs: m' to ~1e-9; second reference level for weights below the fp32 range) when the event
    // hangs on samples the fast one cannot resolve: no weighted sample, W below the fp32 range, or d deep in the window.
    const float z0h = (float)z0, z0l = (float)(z0 - (double)z0h);
    float mx = -INFINITY;
    int jd = 0;
    const float4* rec = P.ev.rec + 2 * s0;
    const int64_t p0 = P.ev.poly_off[ev];
    // samples are sorted in d_L: one of them lies beyond the table iff the last one does
    if (tid == 0 && __float_as_uint(__ldg(rec + 2 * (size_t)(ns - 1)).x) > L.F.tkmax_ev_q) atomicOr(P.flags + l, CHIM_FLAG_TABLE_RANGE);
    bool careful = true;
    if (use_poly && !force_careful) {   // (force_careful: k_events_fast found the unit in need of the careful sweep already)
        if (S.mass_fit) mx = s2_sweep_poly<true>(P.ev.prec_a + p0, P.ev.prec_b + p0, L.F, S.poly, M, ns, zf, wl, jd);
        else mx = s2_sweep_poly<false>(P.ev.prec_a + p0, P.ev.prec_b + p0, L.F, S.poly, M, ns, zf, wl, jd);
        block_argmax(mx, jd, S.kred);
        if (mx > -INFINITY && mx == mx) {
            const float zd = zf[jd];
            float m0 = 0.f, m1 = 0.f, m2 = 0.f, m3 = 0.f;   // W, Q, B, A
            for (int j = tid; j < ns; j += kEvThreads) {
                const float w = ex2f(wl[j] - mx), u = zf[j] - zd;
                wl[j] = w;
                const float we = (j == jd) ? 0.f : w;
                m0 += we;
                m1 = fmaf(we, we, m1);
                const float wu = we * u;
                m2 += wu;
                m3 = fmaf(wu, u, m3);
            }
#pragma unroll
            for (int o = 16; o > 0; o >>= 1) {
                m0 += __shfl_xor_sync(0xffffffffu, m0, o);
                m1 += __shfl_xor_sync(0xffffffffu, m1, o);
                m2 += __shfl_xor_sync(0xffffffffu, m2, o);
                m3 += __shfl_xor_sync(0xffffffffu, m3, o);
            }
            if (lane == 0) { S.red[wid] = m0; S.red[8 + wid] = m1; S.red[16 + wid] = m2; S.red[24 + wid] = m3; }
            __syncthreads();
            if (tid == 0) {
#pragma unroll
                for (int i = 0; i < 4; ++i) {
                    double acc = 0.0;
#pragma unroll
                    for (int k = 0; k < kEvThreads / 32; ++k) acc += S.red[i * 8 + k];
                    S.mom[i] = acc;
                }
                S.slev = 1.0;
                // m2' of the heaviest sample, from its record and the polynomial of 1/(1+z)
                const float4 Ad = __ldg(P.ev.prec_a + p0 + jd);
                float ad = S.poly[2 * kPolyN + 2 * (kPolyN - 2) + 1];
#pragma unroll
                for (int n = kPolyN - 3; n >= 0; --n) ad = fmaf(ad, Ad.z, S.poly[2 * kPolyN + 2 * n + 1]);
                const float mp2d = fmaf(Ad.y, ad, -L.F.mlow_hi);
                // fp32 leaves ~1e-6 (random) + ~5e-7 (the fit, common to all samples) in m2': d ln w = delta/m2'^2 of that.  The
                // careful sweep is taken where this would show in log I: few effective samples (n_eff < neff_min), or all of them deep
                const double neff = (1.0 + S.mom[0]) * (1.0 + S.mom[0]) / (1.0 + S.mom[1]);
                S.careful = (S.mom[0] < 7.9e-31 /* 2^-100 */ || neff < (double)P.neff_min ||
                             (double)mp2d * (double)mp2d < (double)L.F.delta * fmax(0.5 * rsqrt(neff), 0.1)) ? 1 : 0;
            }
            __syncthreads();
            careful = S.careful != 0;
        }
    }
    if (careful) {
        __syncthreads();     // (every thread is done with zf / wl of the fast sweep)
        if (staged && !use_poly) mx = s2_sweep<true>(rec, L.F, rows_s, k_lo, M, ns, z0h, z0l, zf, wl, jd);
        else mx = s2_sweep<false>(rec, L.F, reinterpret_cast<const float4*>(tab), 0, M, ns, z0h, z0l, zf, wl, jd);
        block_argmax(mx, jd, S.kred);
        if (mx > -INFINITY && mx == mx) {
            float l2 = -INFINITY;                       // second reference level: the largest log2 w among the others
            int j2 = 0;
            for (int j = tid; j < ns; j += kEvThreads)
                if (j != jd) l2 = fmaxf(l2, wl[j]);
            block_argmax(l2, j2, S.kred);
            const float zd = zf[jd];
            float m0 = 0.f, m1 = 0.f, m2 = 0.f, m3 = 0.f;   // W'', Q'', B'', A'' relative to l2
            for (int j = tid; j < ns; j += kEvThreads) {
                const float lw = wl[j], u = zf[j] - zd;
                wl[j] = ex2f(lw - mx);                   // what the KDE sees: relative to the heaviest sample
                const float we = (j == jd || !(l2 > -INFINITY)) ? 0.f : ex2f(lw - l2);
                m0 += we;
                m1 = fmaf(we, we, m1);
                const float wu = we * u;
                m2 += wu;
                m3 = fmaf(wu, u, m3);
            }
            double mm[4] = {(double)m0, (double)m1, (double)m2, (double)m3};
            block_sum<kEvThreads, 4>(mm, S.red);
            if (tid == 0) {
                S.mom[0] = mm[0]; S.mom[1] = mm[1]; S.mom[2] = mm[2]; S.mom[3] = mm[3];
                S.slev = (l2 > -INFINITY) ? exp2((double)l2 - (double)mx) : 0.0;
            }
        }
    }
    if (!(mx > -INFINITY)) {   // all-zero event (R15): I = 0
        if (tid == 0) {
            *out = (mx != mx) ? NAN : -INFINITY;
            atomicOr(P.flags + l, CHIM_FLAG_EVENT_ZERO);
            if (P.dbg_h) *P.dbg_h = NAN;
        }
        if (P.dbg_z)
            for (int j = tid; j < ns; j += kEvThreads) {
                const int jo = P.ev.perm[s0 + j];
                P.dbg_z[jo] = z0 + (double)zf[j];
                P.dbg_w[jo] = 0.0;
            }
        return;
    }
    {
        const float zlast = zf[ns - 1];
        const int nsp = (int)ev_ns_pad(ns);
        __syncthreads();     // wl / zf complete (and S.mom published) before the idle slots and the diagnostics read them
        for (int j = ns + tid; j < nsp; j += kEvThreads) {   // idle slots of the last pass sit on the last sample with weight 0
            wl[j] = 0.f;
            zf[j] = zlast;
        }
    }
    if (P.dbg_z)
        for (int j = tid; j < ns; j += kEvThreads) {
            const int jo = P.ev.perm[s0 + j];
            P.dbg_z[jo] = z0 + (double)zf[j];
            P.dbg_w[jo] = (double)wl[j] * exp2((double)mx) * exp(P.ln_shift[ev]);
        }
    const double* zc_g = P.ev.zc + g0;
    const float* qn_g = P.ev.qn + g0;
    // q_g of the first 1024 grid points: requested now, consumed after the bandwidth step (their L2 latency hides behind it)
    float qpre[4];
#pragma unroll
    for (int k = 0; k < 4; ++k) {
        const int g = tid + k * kEvThreads;
        qpre[k] = (g < nz) ? __ldg(qn_g + g) : 0.f;
    }
    const double udz = S.ev_udz;
    const float T = (P.cutoff > 0.0) ? (float)(P.cutoff * sqrt(kHalfLog2e)) : INFINITY;
    if (tid == 0) {   // one thread: bandwidth, and every scalar the pair loop needs
        double h;
        if (P.bw_rule == CHIM_BW_FIXED) {
            h = P.ev.fixed_bw[ev];
        } else {   // Scott on the weighted sample (R3, O7) in the form of R21; sl = 1 unless the careful sweep set a second level
            const double W = S.mom[0], Q = S.mom[1], Bm = S.mom[2], Am = S.mom[3], sl = S.slev;
            const double den = 2.0 * W + sl * (W * W - Q), var = (Am * (1.0 + sl * W) - sl * Bm * Bm) / den;
            const double neff = (1.0 + sl * W) * (1.0 + sl * W) / (1.0 + sl * sl * Q);
            h = (den > 0.0 && var > 0.0) ? sqrt(var) * (double)exp2f(-0.2f * log2f((float)neff)) : NAN;   // fp32 power: dh/h ~ 1e-7 moves log I by ~1e-9
        }
        if (P.dbg_h) *P.dbg_h = h;
        // scaled coordinates x = z' sqrt(log2(e)/2)/h: exp(-d^2/2h^2) = 2^(-dx^2)
        const float scf = (float)(sqrt(kHalfLog2e) / h);
        const double scd = (double)scf;             // samples and grid are scaled by the SAME rounded factor
        const float delta = (float)(udz * scd);
        int Bsel = 0;                                // 0 = direct form
        if (udz > 0.0 && T < INFINITY && (P.kde_method == CHIM_KDE_AUTO || P.kde_method == CHIM_KDE_POWER) && !P.dbg_K) {
            if (delta * 32.f <= 3.3f) Bsel = 32;
            else if (delta * 16.f <= kMaxBlockSpan) Bsel = 16;
        }
        S.h = h; S.scd = scd; S.scf = scf; S.delta = delta; S.xfirst = (float)(S.ev_zfirst * scd); S.Bsel = Bsel;
        // t h below half the (largest) grid spacing: a sample may have no grid point inside its cut-off -> exact evaluation
        S.exact = (P.kde_kernel == CHIM_KERNEL_GAUSS && P.cutoff > 0.0 && h > 0.0 && P.cutoff * h < 0.5 * S.ev_maxdz) ? 1 : 0;
        // local-expansion form: equally spaced grid, a cut-off, boxes of ~1 unit of y = z'/(sqrt(2) h) that fit the stage
        S.le_nbox = 0; S.le_D = 0;
        if (udz > 0.0 && T < INFINITY && P.kde_method == CHIM_KDE_AUTO && !P.dbg_K && h > 0.0 && isfinite(h)) {
            const float scy = (float)(0.70710678118654752440 / h);
            const float dy = (float)(udz * (double)scy);
            const int m = max(1, (int)lrintf(1.0f / dy));
            const float wbox = (float)m * dy, Ty = (float)(P.cutoff * 0.70710678118654752440);
            const float yfirst = (float)(S.ev_zfirst * (double)scy);
            const float fb_lo = floorf((zf[0] * scy - yfirst) / wbox + 0.5f), fb_hi = floorf((zf[ns - 1] * scy - yfirst) / wbox + 0.5f);
            const float fD = ceilf((Ty + 0.5f * wbox) / dy) + 1.0f;
            if (wbox <= kLeMaxW && fb_hi - fb_lo < (float)kLeMaxBox && fabsf(fb_lo) < 1e6f && fabsf(fb_hi) < 1e6f && fD < 1e5f &&
                fabsf(fb_lo) * (float)m < 1e8f && fabsf(fb_hi) * (float)m < 1e8f) {
                const int D = (int)fD, nbox = (int)(fb_hi - fb_lo) + 1;
                // issue-slot estimates (profiles/r01c): coefficient build 1/16 per FMA, evaluation ~1 per sample; power form
                // 2.25 per 64 pairs.  Few samples (many-1d pixels) do not amortise the coefficient build.
                const float le_cost = 0.0625f * (float)nbox * (float)kLeP * (2.f * fD + 1.f) + (float)(P.n_bins > 0 ? P.n_bins : ns) + 150.f;
                const float pw_cost = Bsel ? 0.035f * (float)(P.n_bins > 0 ? P.n_bins : ns) * (2.f * T / delta + (float)Bsel) : INFINITY;
                if (le_cost <= pw_cost && le_bytes(ev_nz_pad(nz), D, nbox) <= ev_aux_bytes(P.ev.max_nz)) {
                    S.scy = scy; S.dy = dy; S.yfirst = yfirst; S.le_m = m; S.le_D = D; S.le_blo = (int)fb_lo; S.le_nbox = nbox;
                }
            }
        }
    }
    __syncthreads();
    if (P.kde_method == CHIM_KDE_NONE) {   // diagnostic: S3 skipped; flat p_gal on a wide grid: I = mean weight (pin P5)
        if (tid == 0) {
            const double sw = 1.0 + S.slev * S.mom[0];     // sum_j w_j / w_d
            *out = log(sw / (double)ns) + (double)mx * 0.69314718055994530942 + P.ln_shift[ev];
        }
        return;
    }
    const double h = S.h;
    if (!(h > 0.0) || !isfinite(h)) {
        if (tid == 0) {
            *out = NAN;
            atomicOr(P.flags + l, CHIM_FLAG_BW_DEGENERATE);
        }
        if (P.dbg_K) for (int g = tid; g < nz; g += kEvThreads) P.dbg_K[g] = NAN;
        return;
    }
    int ns3 = ns;            // samples S3 works on: the pseudo-samples when binning is on
    if (P.n_bins > 0) {
        // Sample binning (R23): n_bins equal-width bins on [z_first, z_last] (sorted samples); a bin becomes
        // one pseudo-sample at the weighted mean redshift of its members with the sum of their weights (empty: weight 0, bin
        // centre).  h and 1/N_s stay those of the original samples.  The pseudo-samples overwrite zf / wl (sorted by
        // construction); bins are accumulated in the stage with shared-memory atomics (order-dependent at the fp32 level).
        const int nb = (zf[ns - 1] > zf[0]) ? P.n_bins : 1;
        float* bw = reinterpret_cast<float*>(aux);
        float* bz = bw + P.n_bins;
        const float zlo = zf[0], width = (zf[ns - 1] - zlo) / (float)nb, inv_width = (nb > 1) ? 1.0f / width : 0.f;
        for (int b = tid; b < nb; b += kEvThreads) { bw[b] = 0.f; bz[b] = 0.f; }
        __syncthreads();
        {   // every thread walks a contiguous run of the (sorted) samples and flushes a bin when the index changes:
            // 2-3 atomics per thread instead of one per sample, and neighbours rarely meet in a bin
            const int chunk = ((ns + kEvThreads - 1) / kEvThreads) | 1;          // odd: spreads the lanes over the banks
            const int j0 = tid * chunk, j1 = min(j0 + chunk, ns);
            int cur = -1;
            float aw = 0.f, az = 0.f;
            for (int j = j0; j < j1; ++j) {
                const float w = wl[j], dz = zf[j] - zlo;
                const int b = min(max((int)(dz * inv_width), 0), nb - 1);
                if (b != cur) {
                    if (aw > 0.f) { atomicAdd(bw + cur, aw); atomicAdd(bz + cur, az); }
                    cur = b; aw = 0.f; az = 0.f;
                }
                aw += w;
                az = fmaf(w, dz, az);
            }
            if (aw > 0.f) { atomicAdd(bw + cur, aw); atomicAdd(bz + cur, az); }
        }
        __syncthreads();
        const int nbp = (int)ev_ns_pad(nb);
        for (int b = tid; b < nbp; b += kEvThreads) {
            const int bb = min(b, nb - 1);
            const float W = bw[bb];
            zf[b] = (W > 0.f) ? zlo + bz[bb] / W : zlo + ((float)bb + 0.5f) * width;
            wl[b] = (b < nb) ? W : 0.f;                          // idle slots of the last pass: last pseudo-sample, weight 0
        }
        __syncthreads();
        ns3 = nb;
    }
    if (P.kde_kernel == CHIM_KERNEL_EPANECHNIKOV) {
        // Epanechnikov kernel (R19), exact on any grid without a pair loop: with the prefix sums
        // Q_k[g] = sum_{g' < g} q_g' z'^k over the event grid,
        //   A_j = sum_{|z_g - z_j| <= hE} q_g (1 - (z_g - z_j)^2 / hE^2) = dQ0 - (dQ2 - 2 z_j dQ1 + z_j^2 dQ0) / hE^2
        // over the index range [a, b] of the support; I = 3/(4 hE N_s) sum_j w_j A_j.  fp64 (the bracket cancels ~1e3).
        // A grid point that rounding puts on the wrong side of the support edge contributes ~1e-16 (the kernel is 0 there).
        const double hE = 2.2360679774997896964 * h, ihE2 = 1.0 / (hE * hE);
        const double* q0 = P.ev.ep_q0 + g0 + ev;
        const double* q1 = P.ev.ep_q1 + g0 + ev;
        const double* q2 = P.ev.ep_q2 + g0 + ev;
        const double zfirst = S.ev_zfirst, idz = (udz > 0.0) ? 1.0 / udz : 0.0;
        double lsum = 0.0;
        for (int j = tid; j < ns3; j += kEvThreads) {
            const double zj = (double)zf[j], lo = zj - hE, hi = zj + hE;
            int a, b;
            if (udz > 0.0) {
                a = (int)fmax(0.0, ceil((lo - zfirst) * idz));
                b = (int)fmin((double)(nz - 1), floor((hi - zfirst) * idz));
            } else {
                int x = 0, y = nz;
                while (x < y) { const int mid = (x + y) >> 1; if (zc_g[mid] < lo) x = mid + 1; else y = mid; }
                a = x;
                y = nz;
                while (x < y) { const int mid = (x + y) >> 1; if (zc_g[mid] <= hi) x = mid + 1; else y = mid; }
                b = x - 1;
            }
            if (b >= a) {
                const double d0 = q0[b + 1] - q0[a], d1 = q1[b + 1] - q1[a], d2 = q2[b + 1] - q2[a];
                const double A = d0 - (d2 - 2.0 * zj * d1 + zj * zj * d0) * ihE2;
                lsum = fma((double)wl[j], fmax(A, 0.0), lsum);
            }
        }
        double t1[1] = {lsum};
        block_sum<kEvThreads, 1>(t1, S.red);
        if (P.dbg_K) for (int g = tid; g < nz; g += kEvThreads) P.dbg_K[g] = NAN;
        if (tid == 0) {
            const double I = t1[0] * 0.75 / ((double)ns * hE);
            if (I > 0.0) *out = log(I) + (double)mx * 0.69314718055994530942 + S.ev_ln_out;
            else if (I == 0.0) { *out = -INFINITY; atomicOr(P.flags + l, CHIM_FLAG_EVENT_ZERO); }
            else *out = NAN;
        }
        return;
    }
    const float scf = S.scf, delta = S.delta, xfirst = S.xfirst;
    const int Bsel = S.Bsel;
    const int nzp = (int)ev_nz_pad(nz);
    const bool on_grid = P.placement == CHIM_ON_GRID;
    const int le_nbox = S.le_nbox;
    LeSmem LM = le_layout(aux, (size_t)nzp, S.le_D, le_nbox);
    if (le_nbox) {            // local-expansion form: plain q_g (x grid factor)
#pragma unroll
        for (int k = 0; k < 4; ++k) {           // the prefetched part
            const int g = tid + k * kEvThreads;
            if (g < nzp) {
                float q = qpre[k];
                if (on_grid && g < nz)
                    q = (float)((double)q * grid_factor(L, P.dc_tab + (size_t)l * (P.n_table + 1 + kZPad), P.n_table + 1 + kZPad,
                                                        P.z_table_max / P.n_table, zc_g[g] + z0));
                LM.qs[g] = q;
            }
        }
        for (int g = tid + 4 * kEvThreads; g < nzp; g += kEvThreads) {
            float q = 0.f;
            if (g < nz) {
                q = qn_g[g];
                if (on_grid)
                    q = (float)((double)q * grid_factor(L, P.dc_tab + (size_t)l * (P.n_table + 1 + kZPad), P.n_table + 1 + kZPad,
                                                        P.z_table_max / P.n_table, zc_g[g] + z0));
            }
            LM.qs[g] = q;
        }
        le_psi_table(LM.psi, S.le_D, S.dy);
    } else if (Bsel && !on_grid) {   // power form: q'_g = q_g 2^(-(b delta)^2), b = g mod B, duplicated for the packed FMA
        for (int g = tid; g < nzp; g += kEvThreads) {   // (the barriers above fenced the last reads of the staged tables)
            const float bd = (float)(g & (Bsel - 1)) * delta;
            gqp[g] = (g < nz) ? qn_g[g] * ex2f(-bd * bd) : 0.f;
        }
    } else {
        const double scd = S.scd;
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
                gqp[g] = q * ex2f(-bd * bd);
            } else {
                gq[g] = make_float2(xg, q);
            }
        }
    }
    __syncthreads();

    // ---- S3 + S4: warp passes over 128 consecutive (sorted) samples ----------------------------------------
    const int n_pass = (ns3 + kPass - 1) / kPass;
    const float inv_delta = (udz > 0.0) ? 1.f / delta : 0.f;
    const float bd = (float)Bsel * delta, inv_bd = Bsel ? 1.f / bd : 0.f;
    const int a_max = Bsel ? nzp / Bsel - 1 : 0;
    double lsum = 0.0;                          // this lane's sum_j w_j A_j
    unsigned long long pairs_exec = 0, pairs_cut = 0;
    if (le_nbox) lsum = le_phase<kStats>(S, LM, zf, wl, ns3, nz, (float)(P.cutoff * 0.70710678118654752440), pairs_exec, pairs_cut);
    else for (;;) {
        int pass = 0;
        if (lane == 0) pass = atomicAdd(&S.pass_counter, 1);
        pass = __shfl_sync(0xffffffffu, pass, 0);
        if (pass >= n_pass) break;
        const int j0 = pass * kPass + lane * 4;
        const float4 zz = *reinterpret_cast<const float4*>(zf + j0);
        const float4 ww = *reinterpret_cast<const float4*>(wl + j0);
        const float w[4] = {ww.x, ww.y, ww.z, ww.w};
        const float x[4] = {zz.x * scf, zz.y * scf, zz.z * scf, zz.w * scf};
        // samples are sorted in z: the pass spans [first, last] (idle slots repeat the last sample)
        const float xa = zf[pass * kPass] * scf, xb = zf[pass * kPass + kPass - 1] * scf;
        const float xmn = fminf(xa, xb), xmx = fmaxf(xa, xb);
        float A[4] = {0.f, 0.f, 0.f, 0.f};
        bool done = false;
        if (Bsel) {
            // (a product with the rounded 1/bd may land one block early or late at an exact block edge: the pairs
            // concerned sit at the cut-off distance, where a Gaussian term is below 2^-26 of the peak)
            const int a_lo = max(0, (int)floorf((xmn - T - xfirst) * inv_bd));
            const int a_hi = min(a_max, (int)floorf((xmx + T - xfirst) * inv_bd));
            // largest exponent of s^b inside a block: 2 |u| delta (B-1) with |u| <= span + T + B delta
            if (2.f * (xmx - xmn + T + bd) * bd <= kMaxPowExp) {
                if (a_hi >= a_lo) {
                    if (Bsel == 32) power_pass<32>(gqp, a_lo, a_hi, xfirst, delta, x, A);
                    else power_pass<16>(gqp, a_lo, a_hi, xfirst, delta, x, A);
                    if (kStats && lane == 0) pairs_exec += (unsigned long long)(a_hi - a_lo + 1) * Bsel * kPass;
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
                    const float xg = fmaf((float)g, delta, xfirst), q = gqp[g] * ex2f(bdg * bdg);
#pragma unroll
                    for (int k = 0; k < 4; ++k) { const float d = xg - x[k]; A[k] = fmaf(q, ex2f(-d * d), A[k]); }
                }
            } else if (P.dbg_K) {
#pragma unroll 1
                for (int g = g_lo; g <= g_hi; ++g) {
                    const float2 v = gq[g];
                    float kv = 0.f;
#pragma unroll
                    for (int k = 0; k < 4; ++k) {
                        const float d = v.x - x[k], e = ex2f(-d * d);
                        A[k] = fmaf(v.y, e, A[k]);
                        kv = fmaf(w[k], e, kv);
                    }
                    double kd = warp_sum((double)kv);
                    if (lane == 0) atomicAdd(P.dbg_K + g, kd);
                }
            } else {
#pragma unroll 2
                for (int g = g_lo; g <= g_hi; ++g) {
                    const float2 v = gq[g];
#pragma unroll
                    for (int k = 0; k < 4; ++k) { const float d = v.x - x[k]; A[k] = fmaf(v.y, ex2f(-d * d), A[k]); }
                }
            }
            if (kStats && lane == 0 && g_hi >= g_lo) pairs_exec += (unsigned long long)(g_hi - g_lo + 1) * kPass;
        }
        lsum += (double)fmaf(w[0], A[0], fmaf(w[1], A[1], fmaf(w[2], A[2], w[3] * A[3])));
        if (kStats) {
            if (udz > 0.0 && T < INFINITY) {   // algorithmic pair count: grid points within the cut-off of each weighted sample
#pragma unroll
                for (int k = 0; k < 4; ++k)
                    if (w[k] > 0.f) {
                        const int a = max(0, (int)ceilf((x[k] - T - xfirst) * inv_delta)), b = min(nz - 1, (int)floorf((x[k] + T - xfirst) * inv_delta));
                        pairs_cut += (unsigned long long)max(0, b - a + 1);
                    }
            } else {
#pragma unroll
                for (int k = 0; k < 4; ++k) pairs_cut += (w[k] > 0.f) ? (unsigned long long)nz : 0ull;
            }
        }
    }
    // K(z) = 1/(N_s h sqrt(2 pi)) sum_j w_j exp(..); the weights were divided by 2^mx
    const double knorm = 1.0 / ((double)ns * h * 2.50662827463100050242);
    const double ln_wscale = (double)mx * 0.69314718055994530942;
    double tot[3] = {lsum, (double)pairs_exec, (double)pairs_cut};
    if constexpr (kStats) {
        block_sum<kEvThreads, 3>(tot, S.red);
        if (tid == 0 && P.stats) {
            if (tot[1] > 0.0) atomicAdd(P.stats, (unsigned long long)tot[1]);
            if (tot[2] > 0.0) atomicAdd(P.stats + 1, (unsigned long long)tot[2]);
        }
    } else {
        double t1[1] = {lsum};
        block_sum<kEvThreads, 1>(t1, S.red);
        tot[0] = t1[0];
    }
    if (P.dbg_K) {   // diagnostics: turn the accumulated sums into K(z_g)
        __syncthreads();
        const double ks = knorm * exp(ln_wscale + P.ln_shift[ev]);
        for (int g = tid; g < nz; g += kEvThreads) P.dbg_K[g] *= ks;
    }
    if ((S.exact || tot[0] == 0.0) && !P.dbg_K) {   // (block-uniform) units outside the reach of the fp32 pair loop
        const double l2s = exact_log2_kde(L, on_grid ? P.dc_tab + (size_t)l * (P.n_table + 1 + kZPad) : nullptr, P.n_table + 1 + kZPad,
                                          P.z_table_max / P.n_table, zf, wl, ns3, zc_g, qn_g, nz, z0, h, S.red, S.kred);
        if (tid == 0) {
            if (l2s > -INFINITY) *out = l2s * 0.69314718055994530942 + log(knorm) + ln_wscale + S.ev_ln_out;
            else { *out = -INFINITY; atomicOr(P.flags + l, CHIM_FLAG_EVENT_ZERO); }
        }
        return;
    }
    if (tid == 0) {
        double I = tot[0] * knorm;
        if (I > 0.0) *out = log(I) + ln_wscale + S.ev_ln_out;
        else if (I == 0.0) { *out = -INFINITY; atomicOr(P.flags + l, CHIM_FLAG_EVENT_ZERO); }
        else *out = NAN;
    }
}

// Grid: (events x lambdas) with lambda fastest [optionally through ev_list: the events k_events_fast does not take], or --
// work-list mode -- a fixed number of CTAs that loop over the units k_events_fast handed over in this batch.
template <bool kStats>
__global__ void __launch_bounds__(kEvThreads, CHIM_EV_BLOCKS) k_events(EventKernelParams P) {
    extern __shared__ __align__(128) unsigned char smem_raw[];
    if (P.worklist) {
        const unsigned n = *P.work_count;
        bool again = false;
        for (unsigned u = blockIdx.x; u < n; u += gridDim.x) {
            const uint32_t entry = P.worklist[u], unit = entry & 0x7FFFFFFFu;     // (bit 31: take the careful sweep at once)
            events_unit<kStats>(P, (int)(unit / (uint32_t)P.ev.n_events), (int)(unit % (uint32_t)P.ev.n_events), smem_raw, again, (entry >> 31) != 0u);
            again = true;
            __syncthreads();
        }
        return;
    }
    int l, ev;
    if (P.dbg_event >= 0) { l = blockIdx.x; ev = P.dbg_event; }
    else {   // lambda fastest: CTAs in flight share an event
        l = blockIdx.x % P.n_lambda;
        ev = blockIdx.x / P.n_lambda;
        if (P.ev_list) ev = P.ev_list[ev];
    }
    events_unit<kStats>(P, l, ev, smem_raw, false, false);
}

int events_mass_stage_rows(int n_mass) { return min(kMassStage, n_mass + 2); }

size_t events_smem_bytes(int max_ns, int max_nz) {
    return ((sizeof(EvSmem) + 127) / 128) * 128 + 2 * sizeof(float) * ev_ns_pad((size_t)max_ns) + ev_aux_bytes((size_t)max_nz);
}

cudaError_t launch_events(const EventKernelParams& P, bool count_pairs, cudaStream_t st) {
    size_t smem = events_smem_bytes(P.ev.max_ns, P.ev.max_nz);
    auto kern = count_pairs ? k_events<true> : k_events<false>;
    cudaError_t e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    if (e != cudaSuccess) return e;
    long long nb = (P.dbg_event >= 0) ? P.n_lambda : (long long)P.n_lambda * (P.ev_list ? P.n_ev_list : P.ev.n_events);
    if (P.worklist) nb = P.worklist_ctas;
    if (nb <= 0) return cudaSuccess;
    kern<<<(unsigned)nb, kEvThreads, smem, st>>>(P);
    return cudaGetLastError();
}

}  // namespace chim
