// chim_internal.cuh -- device-side data layout and shared device functions of libchim.
// Not part of the public ABI (see include/chim.h).  Shares nothing with oracle/.
#pragma once
#include <cuda_runtime.h>
#include <math.h>
#include <stdint.h>

#include "../../include/chim.h"

namespace chim {

constexpr double kCkms = 299792.458;       // speed of light [km/s]
constexpr int kGLWin = 32;                 // Gauss-Legendre nodes for the normalisation integrals (S1)
constexpr int kGLPanel = 8;                // Gauss-Legendre nodes per panel of the window table (S1)
constexpr int kZPad = 32;                  // d_C table panels kept beyond z_table_max (stencil safety)
constexpr double kLnFloor = -1.0e4;        // ln of "zero" in the log-space tables (exp underflows to the 1e-307 floor)
constexpr double kHalfLog2e = 0.72134752044448170368;  // log2(e)/2 : exp(-d^2/2h^2) = 2^(-(d s)^2), s^2 = kHalfLog2e/h^2

// fp32 view of the per-lambda constants used per sample / injection (S2, S5).  Values that enter a difference of
// nearly equal numbers are carried as an unevaluated sum hi + lo of two floats.
struct alignas(16) LamF {
    // the 16 constants of poly_sample first, as four 16-byte groups (k_events_fast / k_inject read them with four loads)
    float mlow_hi;            // m_low (leading float)
    float tm_scale;           // mass-table coordinate tm = ln(m1) tm_scale + mlow_tm, clamped to [1, tm_max]
    float mlow_tm;            // 1 - ln(m_low) tm_scale
    float mhigh_p;            // m_high - m_low
    float beta2;              // beta log2(e)
    float delta;              // delta_m
    float win_lo, win_hi;     // clamp of m' strictly inside the smoothing window
    float two_dl2e, d2l2e;    // 2 delta log2(e), delta^2 log2(e): log2(e) f = (two_dl2e m' - d2l2e) / (m' (m' - delta))
    float gk2, cpsi;          // (gamma + kappa) log2(e) and gk2 ln(1 + z_p): log2 psi = gamma2 u - log2(1 + 2^(gk2 u - cpsi));
                              // placement ON_GRID (no psi in the sample weights): gk2 = 0, cpsi = 100
    float tm_max;
    float gk2_inj, cpsi_inj;  // gk2, cpsi for the injections (psi is always in s_j)
    float beta2_lo;           // beta log2(e) - beta2 (used by the table path, sample_eval; the polynomial sweeps take beta2 alone: measured,
                              // the extra FMA per sample costs 3 % of k_events_fast for < 1e-7 in log I -- DESIGN.md sec. 7)
    // the rest (table path, hi + lo pairs)
    float mlow_lo;            // m_low - mlow_hi
    float lm0_hi, lm0_lo;     // ln m_low (origin of the mass table)
    float tm_one;             // 1 + tm_shift (LamConst): the table path's coordinate (ln m1 - lm0) tm_scale + tm_one addresses the same shifted nodes
    float tkmax_ev, tkmax_inj;// table coordinate beyond which z > z_table_max
    float zcat_hi, zcat_lo;   // z_cat_max (R6) as hi + lo
    uint32_t tkmax_ev_q;      // tkmax_ev in the 12.20 fixed point of the event records
};
// the first 64 bytes of LamF through four 128-bit loads
__device__ __forceinline__ void load_lamf_hot(LamF& F, const LamF* __restrict__ g) {
    const float4* q = reinterpret_cast<const float4*>(g);
    const float4 a = __ldg(q), b = __ldg(q + 1), c = __ldg(q + 2), d = __ldg(q + 3);
    F.mlow_hi = a.x; F.tm_scale = a.y; F.mlow_tm = a.z; F.mhigh_p = a.w;
    F.beta2 = b.x; F.delta = b.y; F.win_lo = b.z; F.win_hi = b.w;
    F.two_dl2e = c.x; F.d2l2e = c.y; F.gk2 = c.z; F.cpsi = c.w;
    F.tm_max = d.x; F.gk2_inj = d.y; F.cpsi_inj = d.z; F.beta2_lo = d.w;
}

// Per-lambda constants written by the table kernel (S1), read by every other kernel.
struct LamConst {
    double H0, Om, Xi0, n, alpha, beta, delta, m_low, m_high, mu, sigma, lg, gamma, kappa, zp;
    double c_H0;        // c / H0 [Mpc]
    double m_c;         // m_low + delta_m (upper end of the smoothing window)
    double a_pl;        // ln[(1 - lambda_g) / (N_pl Z1)]   (power-law prefactor incl. 1/Z1)
    double a_g;         // ln[lambda_g / (sigma_g sqrt(2 pi) Z1)]
    double inv2s2;      // 1 / (2 sigma_g^2)
    double W_c;         // int_{m_low}^{m_c} m^beta S(m) dm
    double bp1;         // beta + 1
    double inv_bp1;     // 1 / (beta + 1)
    double pow_mc_bp1;  // m_c^(beta+1)
    double ln_mc;       // ln m_c
    double gk;          // gamma + kappa
    double ln1pzp;      // ln(1 + z_p)
    double vol_norm;    // 3 / d_C(z_cat_max)^3 : u(z) = d_C^2 (c/H0/E) * vol_norm   (R6)
    double tkmax_ev;    // samples with table coordinate tk > tkmax have z > z_table_max (weight 0)
    double tkmax_inj;
    double dl_tabmax;   // d_L^gw(z_table_max)
    double Z1;          // normalisation of p(m1)
    double win_scale;   // n_win / delta_m
    double inv_delta;   // 1 / delta_m
    double lm0;         // mass table: node coordinate tm = (ln m1 - lm0) * inv_dlm + 1
    double inv_dlm;
    double tm_shift;    // (float)mlow_tm - (1 - lm0 inv_dlm): the rounding of LamF::mlow_tm in table rows; the nodes of the mass table are
                        // shifted by it, so the fp32 coordinate ln m1 * tm_scale + mlow_tm of the sample kernels is exact
    uint32_t flags;     // CHIM_FLAG_LAMBDA_DOMAIN | CHIM_FLAG_DL_NONMONOTONE
    int32_t beta_is_m1; // |beta + 1| < 1e-12 : log form of the power integral
    LamF F;             // fp32 constants of the sample kernels (S2, S5)
};

// One interval of the per-lambda interpolation table in x = ln d_L, local coordinate t in [0,1), fp32 (64 B):
//   z(t) = z_hi + (z_lo + t (z1 + t (z2 + t z3)))      redshift: cubic through 4 nodes, leading term as hi + lo
//   a(t) = a_hi + (a_lo + t (a1 + t (a2 + t a3)))      1/(1+z), same form (feeds the difference m^d a - m_low)
//   u(t) = u0 + t (u1 + t u2)                           ln(1+z): the cubic with t^3 economised (Chebyshev) away
//   r(t) = r0 + t (r1 + t r2)                           log2 of the smooth redshift factor of the weight
// (events: psi/J or 1; injections: psi u_vol / J).
struct __align__(16) Row {
    float z_hi, z_lo, z1, z2;
    float z3, a_hi, a_lo, a1;
    float a2, a3, u0, u1;
    float u2, r0, r1, r2;
};

// Geometry of a ln d_L table: sample coordinate tk = (ln dL - x0)/dx + 1, interval k = floor(tk) in [1, K],
// nodes idx = 0..K+2 at x = x0 + (idx-1) dx, rows stored for k = 0..K+1 (rows 0 and K+1 are never addressed
// by an in-range sample).
struct DlGrid {
    double x0, dx;
    int32_t K;  // number of intervals; 0 = table absent
    __host__ __device__ int rows() const { return K + 2; }
};

struct TableParams {
    double z_table_max, z_cat_max;
    int32_t n_table, n_win, placement;
    int32_t n_mass;      // intervals of the per-lambda mass table (in ln m1)
    double ln_m_top;     // ln of the largest detector-frame m1 of the loaded sets (upper end of the mass table)
    DlGrid ev, inj;
};

// One interval of the per-lambda mass table in y = ln m1 (local coordinate t in [0,1]): cubic c0 + t(c1 + t(c2 + t c3)),
// fp32, of  LQ2 = log2[ p(m1)/S(m1) * m1'^2 S(m1)/C(m1) ],  m1' = m1 - m_low  -- i.e. log2 of p(m1)/C(m1) m1'^2,
// smooth and finite on [m_low, inf) because C/S ~ rho m1'^2 (M3/M4).  Two variants per lambda, stored as two
// consecutive arrays of n_mass + 2 rows: "a" with the power law present (m1 <= m_high), "b" the Gaussian only.
typedef float4 MassRow;

// Packed, lambda-independent record of one posterior sample / injection (32 B = {A, B}, read with one 256-bit load).
//   events:     A = {tkq, m1d_hi, m1d_lo, m2d_hi}   B = {m2d_lo, ln m1d, ln(m2d/m1d), log2(1/prior) - event scale}
//               tkq = table coordinate in 12.20 fixed point (interval in the upper 12 bits)
//   injections: A = {k, t, m1d, m2d}                B = {ln m1d, ln(m2d/m1d), log2(1/p_draw) - set scale, 0}
//               (t kept as a full float: the support cut z <= z_cat_max of R6 is a step)
constexpr int kTkFracBits = 20;
constexpr int kMaxDlRows = (1 << (32 - kTkFracBits)) - 3;   // largest n_dl_table the fixed-point coordinate can address

__device__ __forceinline__ float ex2f(float x) {
    float y;
    asm("ex2.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x));
    return y;
}
__device__ __forceinline__ float lg2f(float x) {
    float y;
    asm("lg2.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x));
    return y;
}
__device__ __forceinline__ float rcpf(float x) {
    float y;
    asm("rcp.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x));
    return y;
}

// 2^y as a double for any float y (the fp32 exponent range is not enough for injection weights carrying an arbitrary
// draw-density scale): integer part through the exponent field, fraction through MUFU.EX2.  y = -inf gives 0.
__device__ __forceinline__ double ex2_to_double(float y) {
    const float yc = fminf(fmaxf(y, -1000.f), 1000.f);
    const float ti = yc + 12582912.f;                   // 1.5 * 2^23: round to nearest integer
    const int n = __float_as_int(ti) - 0x4B400000;
    const float e = ex2f(yc - (ti - 12582912.f));       // in [0.70, 1.42]
    const double ed = (double)e;
    const double v = __hiloint2double(__double2hiint(ed) + (n << 20), __double2loint(ed));
    return (y > -1000.f) ? v : 0.0;
}

// Records of the local-polynomial sweeps, split for 24 B per sample: A = {m1d, m2d, t, ln m1d}, B = {ln m2d, log2(1/prior)}
// (the masses first: they enter one packed FMA, and a 128-bit load fills aligned register pairs)
struct PRec { float4 A; float2 B; };
__device__ __forceinline__ PRec ldg_stream_prec(const float4* pa, const float2* pb) {   // streaming reads (once per CTA)
    PRec r;
    asm volatile("ld.global.nc.L1::no_allocate.v4.f32 {%0,%1,%2,%3}, [%4];" : "=f"(r.A.x), "=f"(r.A.y), "=f"(r.A.z), "=f"(r.A.w) : "l"(pa));
    asm volatile("ld.global.nc.L1::no_allocate.v2.f32 {%0,%1}, [%2];" : "=f"(r.B.x), "=f"(r.B.y) : "l"(pb));
    return r;
}

// Where a thread finds the per-lambda mass table: rows [lo, lo + cap) of both variants staged in shared memory
// (variant "b" at offset cap), everything else in global memory.
struct MassLookup {
    const MassRow* g;          // [2][n_mass + 2] rows of this lambda
    const MassRow* s;          // staged rows or null
    int lo, cap, n_mass;
};

// The two halves separately, for the doubly prefetched sweeps (k_events_fast, k_inject).  Half A is first touched at the top of
// a sample and dead after its polynomials, so its next load may move up into the sample; half B enters a sample's last two
// operations (poly_sample), and `after` (any value computed from them) pins the load of the NEXT B behind them -- otherwise the
// compiler issues it early into a second register pair and copies it over later, and that copy waits for the load.
__device__ __forceinline__ float4 ldg_stream_a(const float4* pa) {
    float4 r;
    asm volatile("ld.global.nc.L1::no_allocate.v4.f32 {%0,%1,%2,%3}, [%4];" : "=f"(r.x), "=f"(r.y), "=f"(r.z), "=f"(r.w) : "l"(pa));
    return r;
}
__device__ __forceinline__ void ldg_stream_b(float2& r, const float2* pb, float after) {
    // (predicated on `after` being a number or +-inf -- a true dependency the assembler cannot remove; a NaN weight leaves the
    // previous values in place, and its unit is not-a-number anyway)
    asm volatile("{\n .reg .pred p;\n setp.le.f32 p, %3, 0f7F800000;\n @p ld.global.nc.L1::no_allocate.v2.f32 {%0,%1}, [%2];\n}"
                 : "+f"(r.x), "+f"(r.y)
                 : "l"(pb), "f"(after));
}

struct Rec { float4 A, B; };   // one packed record (32 B, 32-byte aligned)
__device__ __forceinline__ Rec ldg_stream_rec(const float4* p) {   // streaming 256-bit read (read once per CTA)
    Rec r;
    asm volatile("ld.global.nc.L1::no_allocate.v8.f32 {%0,%1,%2,%3,%4,%5,%6,%7}, [%8];"
                 : "=f"(r.A.x), "=f"(r.A.y), "=f"(r.A.z), "=f"(r.A.w), "=f"(r.B.x), "=f"(r.B.y), "=f"(r.B.z), "=f"(r.B.w)
                 : "l"(p));
    return r;
}

// Steps S2 / S5 for one sample (or injection): redshift from the table, source-frame masses, log2 of the weight
//   w = p(m1, m2 | lambda_m) * R(z) / prior,   p(m1,m2) = p(m1) m2^beta S(m2) / C(m1)     (M1-M4)
//   log2 w = LQ2(ln m1) + beta log2 m2 + log2 R + log2(1/prior) - 2 log2 m1' - log2(1 + e^f(m2'))
//   LQ2  per-lambda mass table (MassRow): log2[p(m1)/C(m1) m1'^2], smooth on [m_low, inf)
//   S(m2) = 1/(1 + exp(delta/m2' + delta/(m2' - delta))) inside the window, 1 above (M1)
//   log2 R, z, ln(1+z), 1/(1+z): the four polynomials of the sample's row of the z(ln d_L) table
//   PAPER.md:52 (d_L -> z, m = m^d/(1+z)), :195-198 eq. 20 (mass model), :226 eq. 21, :75 eq. 11.
// All fp32; differences of nearly equal numbers (z - z_ref, m^d a - m_low) are formed from hi + lo pairs, so the
// rounding errors left are ~1e-7 relative, independent from sample to sample.  Five MUFU ops
// (rcp, ex2, 2 lg2 here; the final ex2 is the caller's), no fp64, no data-dependent branch except the (rare)
// fall-back of the mass row to global memory.  Returns z - z_ref and log2 w (-inf: weight 0).
// Warp-collective: all 32 lanes must call it together (the rare paths are taken per warp, by vote).
__device__ __forceinline__ void sample_eval(const LamF& F, const float4 q0, const float4 q1, const float4 q2,
                                            const float4 q3, const float t, const float zref_hi, const float zref_lo,
                                            const float m1h, const float m1l, const float m2h, const float m2l,
                                            const float lnm1d, const float lnq, const float ipr2,
                                            const MassLookup& M, const bool in_range, float& zc, float& l2w) {
    // row: q0 = {z_hi, z_lo, z1, z2}  q1 = {z3, a_hi, a_lo, a1}  q2 = {a2, a3, u0, u1}  q3 = {u2, r0, r1, r2}
    zc = (q0.x - zref_hi) + fmaf(fmaf(fmaf(q1.x, t, q0.w), t, q0.z), t, q0.y - zref_lo);
    const float a_hi = q1.y;
    const float a_lo = fmaf(fmaf(fmaf(q2.y, t, q2.x), t, q1.w), t, q1.z);
    const float u = fmaf(fmaf(q3.x, t, q2.w), t, q2.z);
    const float r = fmaf(fmaf(q3.w, t, q3.z), t, q3.y);
    // m' = m^d a - m_low for both masses: exact product + low-order terms
    const float p1 = __fmul_rn(m1h, a_hi), p2 = __fmul_rn(m2h, a_hi);   // never contracted into an FMA
    const float c1 = fmaf(m1h, a_lo, fmaf(m1l, a_hi, fmaf(m1h, a_hi, -p1) - F.mlow_lo));
    const float c2 = fmaf(m2h, a_lo, fmaf(m2l, a_hi, fmaf(m2h, a_hi, -p2) - F.mlow_lo));
    const float mp1 = (p1 - F.mlow_hi) + c1, mp2 = (p2 - F.mlow_hi) + c2;
    const float lm1 = lnm1d - u, lm2 = lm1 + lnq;
    // mass table: coordinate, interval by the magic-number floor, cubic
    float tm = fmaf((lm1 - F.lm0_hi) - F.lm0_lo, F.tm_scale, F.tm_one);
    tm = fminf(fmaxf(tm, 1.0f), F.tm_max);
    const float ti = (tm - 0.5f) + 12582912.f;
    const int km = __float_as_int(ti) - 0x4B400000;
    const float tf = tm - (ti - 12582912.f);
    const bool gauss_only = mp1 > F.mhigh_p;
    const int ks = km - M.lo;
    const bool staged = (unsigned)ks < (unsigned)M.cap;
    float4 c = M.s[(staged ? ks : 0) + (gauss_only ? M.cap : 0)];
    if (__any_sync(0xffffffffu, !staged)) {            // rare: a source mass outside the staged rows
        if (!staged) c = __ldg(M.g + km + (gauss_only ? M.n_mass + 2 : 0));
    }
    float l = fmaf(fmaf(fmaf(c.w, tf, c.z), tf, c.y), tf, c.x);
    l += fmaf(F.beta2, lm2, fmaf(F.beta2_lo, lm2, r + ipr2));
    l = fmaf(-2.f, lg2f(fmaxf(mp1, 1e-30f)), l);
    // smoothing of m2 (M1): log2(e) f = (2 delta m' - delta^2) log2(e) / (m' (m' - delta)), m' clamped inside the window
    if (__any_sync(0xffffffffu, mp2 < F.delta)) {      // skipped by warps whose secondaries all lie above the window
        const float mc = fminf(fmaxf(mp2, F.win_lo), F.win_hi);
        const float f2 = fmaf(F.two_dl2e, mc, -F.d2l2e) * rcpf(mc * (mc - F.delta));
        const float ls = (f2 > 64.f) ? f2 : lg2f(1.0f + ex2f(f2));   // deep in the window 2^f2 overflows; log2(1 + 2^f) = f there
        l -= (mp2 < F.delta) ? ls : 0.f;
    }
    const bool ok = in_range && (mp2 > 0.f);           // R15 support: m_low < m2 (<= m1)
    l2w = ok ? l : -INFINITY;
}

// ---- packed fp32x2 arithmetic (FFMA2 pipe) --------------------------------------------------------------
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
__device__ __forceinline__ f32x2 mul2(f32x2 a, f32x2 b) {
    f32x2 d;
    asm("mul.rn.f32x2 %0, %1, %2;" : "=l"(d) : "l"(a), "l"(b));
    return d;
}
__device__ __forceinline__ f32x2 add2(f32x2 a, f32x2 b) {
    f32x2 d;
    asm("add.rn.f32x2 %0, %1, %2;" : "=l"(d) : "l"(a), "l"(b));
    return d;
}

// ---- local polynomials in ln d_L (S2 of narrow events, S5 of injection chunks) -------------------------------
// Over a range of <= 0.9 in ln d_L, z - z_ref, u = ln(1+z), a = 1/(1+z) and the smooth part r of log2 of the redshift factor
// are polynomials in t in [-1, 1] (degree 6, 5, 5, 6; errors < 1e-8, 4e-8, 6e-8, 1e-9), fitted per (range, lambda)
// through 7 Chebyshev nodes read from the per-lambda z(ln d_L) table.  The Madau-Dickinson turnover of psi is NOT in r
// (its poles sit too close to the real axis for a low degree): it is evaluated per sample from u.
constexpr int kPolyN = 7;
constexpr int kPolyMatDoubles = kPolyN + 2 * kPolyN * kPolyN;   // nodes[7], m7[7][7] (degree 6), m6[7][7] (degree 5, row 6 = 0)

// Coefficients paired for FFMA2: zr[n] = (z_n, r_n), ua[n] = (u_n, a_n); z and r of degree 6, u and a of degree 5.
struct PolyCoef { f32x2 zr[kPolyN], ua[kPolyN - 1]; };
__device__ __forceinline__ void load_poly(PolyCoef& C, const float* __restrict__ pc) {   // pc: float2 zr[7], float2 ua[7]
    const f32x2* q = reinterpret_cast<const f32x2*>(pc);
#pragma unroll
    for (int n = 0; n < kPolyN; ++n) C.zr[n] = q[n];
#pragma unroll
    for (int n = 0; n < kPolyN - 1; ++n) C.ua[n] = q[kPolyN + n];
}

// One segment of eight lanes per fit (four fits per warp; all 32 lanes call it, `valid` says whether the segment's item exists):
// lanes 0..6 of the segment read the table at the Chebyshev nodes of [tk_c - tk_h, tk_c + tk_h] (table coordinates; fp64 from the
// rows' hi + lo terms), then lane n < 7 forms coefficient n of the four polynomials; out[4][7] floats.
//   r = table r + log2(1 + 2^(gk2 u - cpsi)) - beta2 u   (turnover taken out, -beta ln(1+z) of m2^beta folded in)
__device__ __forceinline__ void fit_polys(const LamConst& L, const Row* __restrict__ tab, int K, double tk_c, double tk_h,
                                          double z_ref, bool turn_on, const double* __restrict__ pm, float* __restrict__ out, bool valid,
                                          double* r0_lo = nullptr) {
    const int lane = threadIdx.x & 7;
    double v0 = 0.0, v1 = 0.0, v2 = 0.0, v3 = 0.0;
    if (valid && lane < kPolyN) {
        const double tk = tk_c + tk_h * __ldg(pm + lane);
        const int k = max(1, min((int)tk, K));
        const float t = (float)(tk - (double)k);
        const float4* r = reinterpret_cast<const float4*>(tab + k);
        const float4 q0 = __ldg(r), q1 = __ldg(r + 1), q3 = __ldg(r + 3);
        const double z = (double)q0.x + (double)fmaf(fmaf(fmaf(q1.x, t, q0.w), t, q0.z), t, q0.y);
        const double rr = (double)fmaf(fmaf(q3.w, t, q3.z), t, q3.y);
        const double u = log1p(z);
        const double turn = turn_on ? log2(1.0 + exp2(1.4426950408889634074 * L.gk * (u - L.ln1pzp))) : 0.0;
        v0 = z - z_ref;
        v1 = u;
        v2 = 1.0 / (1.0 + z);
        v3 = rr + turn - 1.4426950408889634074 * L.beta * u;
    }
    double c0 = 0.0, c1 = 0.0, c2 = 0.0, c3 = 0.0;
    const int n = min(lane, kPolyN - 1);
    const double* m7 = pm + kPolyN + n * kPolyN;
    const double* m6 = m7 + kPolyN * kPolyN;
#pragma unroll
    for (int k = 0; k < kPolyN; ++k) {
        const double a7 = __ldg(m7 + k), a6 = __ldg(m6 + k);
        c0 = fma(a7, __shfl_sync(0xffffffffu, v0, k, 8), c0);
        c1 = fma(a6, __shfl_sync(0xffffffffu, v1, k, 8), c1);
        c2 = fma(a6, __shfl_sync(0xffffffffu, v2, k, 8), c2);
        c3 = fma(a7, __shfl_sync(0xffffffffu, v3, k, 8), c3);
    }
    if (valid && lane < kPolyN) {        // out: float2 zr[7] = (z_n, r_n), float2 ua[7] = (u_n, a_n)
        out[2 * lane] = (float)c0;
        out[2 * lane + 1] = (float)c3;
        // r_0 is a factor 2^r_0 common to every weight of the item: its rounding to a float (|r_0| ~ 20: up to 1e-6) does not
        // average out over the samples.  The residual goes back to the caller, who applies it once per item in fp64.
        if (lane == 0 && r0_lo) *r0_lo = c3 - (double)(float)c3;
        out[2 * kPolyN + 2 * lane] = (float)c1;
        out[2 * kPolyN + 2 * lane + 1] = (float)c2;
    }
}

// Steps S2 / S5 for one sample with the local polynomials: the same quantities as sample_eval.  Record
// A = {m1d, m2d, t, ln m1d}, B = {ln m2d, log2(1/prior or 1/p_draw) - scale, .., ..}:
//   m' = m^d a - m_low;  log2 w = LQ2(ln m1) + beta2 ln m2^d + r + B.y - 2 log2 m1' - log2(1 + 2^(gk2 u - cpsi)) - log2(1 + e^f(m2'))
// PAPER.md:52, :195-198 eq. 20, :226 eq. 21, :75 eq. 11.  Warp-collective like sample_eval.
template <bool kFit, bool kTurn = true, bool kWinS = false>
__device__ __forceinline__ void poly_sample(const LamF& F, const float gk2, const float cpsi, const PolyCoef& C, const float4 A,
                                            const float2 Bq, const MassLookup& M, const float tm_lo, const float tm_hi,
                                            float& zc, float& l2w, float& mp2, const float4* __restrict__ win_s = nullptr) {
    const f32x2 t2 = pack2(A.z, A.z);
    f32x2 zr = C.zr[6], ua = C.ua[5];
#pragma unroll
    for (int n = 5; n >= 0; --n) zr = fma2(zr, t2, C.zr[n]);
#pragma unroll
    for (int n = 4; n >= 0; --n) ua = fma2(ua, t2, C.ua[n]);
    float r, u, a, mp1;
    unpack2(zr, zc, r);
    unpack2(ua, u, a);
    unpack2(fma2(pack2(A.x, A.y), pack2(a, a), pack2(-F.mlow_hi, -F.mlow_hi)), mp1, mp2);   // m' = m^d a - m_low
    const float lm1 = A.w - u;
    float tm = fmaf(lm1, F.tm_scale, F.mlow_tm);
    tm = fminf(fmaxf(tm, tm_lo), tm_hi);
    const float ti = (tm - 0.5f) + 12582912.f;
    const int km = __float_as_int(ti) - 0x4B400000;
    const float tf = tm - (ti - 12582912.f);
    const bool gauss_only = mp1 > F.mhigh_p;
    const int ks = km - M.lo;
    float4 c;
    if (kFit) {
        c = M.s[ks + (gauss_only ? M.cap : 0)];
    } else {
        const bool staged = (unsigned)ks < (unsigned)M.cap;
        c = M.s[(staged ? ks : 0) + (gauss_only ? M.cap : 0)];
        if (__any_sync(0xffffffffu, !staged)) {
            if (!staged) c = __ldg(M.g + km + (gauss_only ? M.n_mass + 2 : 0));
        }
    }
    float l = fmaf(fmaf(fmaf(c.w, tf, c.z), tf, c.y), tf, c.x) + r;
    l = fmaf(-2.f, lg2f(mp1), l);            // m1' <= 0 implies m2' <= 0: discarded below
    if (kTurn) l -= lg2f(1.0f + ex2f(fmaf(gk2, u, -cpsi)));   // overflow -> l = -inf, the limit (psi -> 0).  !kTurn: the turnover is part of r
    if (__any_sync(0xffffffffu, mp2 < F.delta)) {
        // (kWinS: the four window constants {win_lo, win_hi, two_dl2e, d2l2e} from shared memory instead of registers)
        const float4 wc = kWinS ? *win_s : make_float4(F.win_lo, F.win_hi, F.two_dl2e, F.d2l2e);
        const float mc = fminf(fmaxf(mp2, wc.x), wc.y);
        const float f2 = fmaf(wc.z, mc, -wc.w) * rcpf(mc * (mc - F.delta));
        const float ls = (f2 > 64.f) ? f2 : lg2f(1.0f + ex2f(f2));   // deep in the window 2^f2 overflows; log2(1 + 2^f) = f there
        l -= (mp2 < F.delta) ? ls : 0.f;
    }
    // the B half of the record enters last (both terms depend on everything above): a streamed record is first touched as late
    // as possible, which is what the prefetch distance of the sweeps is measured against
    l = fmaf(F.beta2, Bq.x, l) + Bq.y;
    l2w = (mp2 > 0.f) ? l : -INFINITY;      // R15 support: m_low < m2
}
template <bool kFit>
__device__ __forceinline__ void poly_sample(const LamF& F, const float gk2, const float cpsi, const PolyCoef& C, const float4 A,
                                            const float2 Bq, const MassLookup& M, const float tm_lo, const float tm_hi,
                                            float& zc, float& l2w) {
    float mp2;
    poly_sample<kFit>(F, gk2, cpsi, C, A, Bq, M, tm_lo, tm_hi, zc, l2w, mp2);
}

// The same sample in two halves, for the sweeps that stream their records through registers (k_events_fast, k_inject).  The head
// consumes the record (both halves) and leaves seven numbers; the tail needs no record.  A sweep runs the heads of two samples,
// requests the records of the next two (one group of loads: ptxas puts every global load of a loop on one scoreboard, so
// waiting for the oldest load waits for the newest -- the group must be the only one in flight and as old as possible at the
// next head), then the two tails.
struct PolyMid {
    float zc, rb, u, mp1, mp2, tf;   // z - z_ref; r + beta2 ln m2d + log2(1/prior); ln(1+z); m1', m2'; fraction of the mass-table row
    int row;                         // staged row of the mass table (variant folded in)
};
__device__ __forceinline__ void poly_head(const LamF& F, const PolyCoef& C, const float4 A, const float2 Bq, const MassLookup& M,
                                          const float tm_lo, const float tm_hi, PolyMid& m) {
    const f32x2 t2 = pack2(A.z, A.z);
    f32x2 zr = C.zr[6], ua = C.ua[5];
#pragma unroll
    for (int n = 5; n >= 0; --n) zr = fma2(zr, t2, C.zr[n]);
#pragma unroll
    for (int n = 4; n >= 0; --n) ua = fma2(ua, t2, C.ua[n]);
    float r, a;
    unpack2(zr, m.zc, r);
    unpack2(ua, m.u, a);
    unpack2(fma2(pack2(A.x, A.y), pack2(a, a), pack2(-F.mlow_hi, -F.mlow_hi)), m.mp1, m.mp2);   // m' = m^d a - m_low
    float tm = fmaf(A.w - m.u, F.tm_scale, F.mlow_tm);
    tm = fminf(fmaxf(tm, tm_lo), tm_hi);
    const float ti = (tm - 0.5f) + 12582912.f;
    m.tf = tm - (ti - 12582912.f);
    m.row = (__float_as_int(ti) - 0x4B400000) - M.lo + ((m.mp1 > F.mhigh_p) ? M.cap : 0);
    m.rb = r + fmaf(F.beta2, Bq.x, Bq.y);
}
template <bool kTurn, bool kWinS>
__device__ __forceinline__ float poly_tail(const LamF& F, const float gk2, const float cpsi, const MassLookup& M, const PolyMid& m,
                                           const float4* __restrict__ win_s) {
    const float4 c = M.s[m.row];
    float l = fmaf(fmaf(fmaf(c.w, m.tf, c.z), m.tf, c.y), m.tf, c.x) + m.rb;
    l = fmaf(-2.f, lg2f(m.mp1), l);          // m1' <= 0 implies m2' <= 0: discarded below
    if (kTurn) l -= lg2f(1.0f + ex2f(fmaf(gk2, m.u, -cpsi)));
    if (__any_sync(0xffffffffu, m.mp2 < F.delta)) {
        float4 wc;
        if (kWinS) {   // (a shared-space load: measured 9.33 against 9.49 ms per step for the generic form)
            asm volatile("ld.shared.v4.f32 {%0,%1,%2,%3}, [%4];" : "=f"(wc.x), "=f"(wc.y), "=f"(wc.z), "=f"(wc.w) : "r"((uint32_t)__cvta_generic_to_shared(win_s)));
        } else wc = make_float4(F.win_lo, F.win_hi, F.two_dl2e, F.d2l2e);
        const float mc = fminf(fmaxf(m.mp2, wc.x), wc.y);
        const float f2 = fmaf(wc.z, mc, -wc.w) * rcpf(mc * (mc - F.delta));
        const float ls = (f2 > 64.f) ? f2 : lg2f(1.0f + ex2f(f2));
        l -= (m.mp2 < F.delta) ? ls : 0.f;
    }
    return (m.mp2 > 0.f) ? l : -INFINITY;    // R15 support: m_low < m2
}
// The records of the next two blocks into R0 / R1, behind the heads that consumed the previous ones (`a0`, `a1`: a value from
// each head; the predicate is a true dependency the assembler cannot remove -- always true for numbers).
__device__ __forceinline__ void ldg_stream_pair_after(PRec& R0, PRec& R1, const float4* pa0, const float2* pb0, const float4* pa1,
                                                      const float2* pb1, float a0, float a1) {
    asm volatile(
        "{\n .reg .pred p;\n setp.le.f32 p, %16, 0f7F800000;\n setp.le.and.f32 p, %17, 0f7F800000, p;\n"
        " @p ld.global.nc.L1::no_allocate.v4.f32 {%0,%1,%2,%3}, [%12];\n"
        " @p ld.global.nc.L1::no_allocate.v2.f32 {%4,%5}, [%13];\n"
        " @p ld.global.nc.L1::no_allocate.v4.f32 {%6,%7,%8,%9}, [%14];\n"
        " @p ld.global.nc.L1::no_allocate.v2.f32 {%10,%11}, [%15];\n}"
        : "+f"(R0.A.x), "+f"(R0.A.y), "+f"(R0.A.z), "+f"(R0.A.w), "+f"(R0.B.x), "+f"(R0.B.y), "+f"(R1.A.x), "+f"(R1.A.y), "+f"(R1.A.z),
          "+f"(R1.A.w), "+f"(R1.B.x), "+f"(R1.B.y)
        : "l"(pa0), "l"(pb0), "l"(pa1), "l"(pb1), "f"(a0), "f"(a1));
}

// k_events_fast: eight warps, each on a contiguous chunk of the event's (d_L-sorted) samples; chunks are whole blocks of 32
// samples, the evaluation takes them in passes of 128
constexpr int kFastWarps = 8;            // (the largest; small sample sets run with four)
constexpr int kFastPass = 128;
__host__ __device__ inline int fast_chunk(int ns, int warps) { return ((ns + warps * 32 - 1) / (warps * 32)) * 32; }   // whole blocks of 32
// Two classes of events, each with its own launch: short sample lists (many-1d pixels) run four warps per CTA and more CTAs per
// SM -- their phases between the barriers are latency-bound -- long ones eight.  Half-width cap of the psi table per class:
// fine grids get a wider table, short lists (wider kernels relative to the grid) a narrower stage.
#ifndef CHIM_FAST_SMALL_NS
#define CHIM_FAST_SMALL_NS 2048
#endif
#ifndef CHIM_FAST_TINY_NS
#define CHIM_FAST_TINY_NS 896
#endif
constexpr int kFastSmallNs = CHIM_FAST_SMALL_NS, kFastTinyNs = CHIM_FAST_TINY_NS;
constexpr int kFastClasses = 3;            // 2, 4, 8 warps
__host__ inline int fast_warps_for(int ns) { return ns <= kFastTinyNs ? 2 : (ns <= kFastSmallNs ? 4 : 8); }
__host__ inline int fast_max_d_for(int warps, int max_nz) { return max_nz > 2048 ? 384 : (warps < 8 ? 160 : 256); }

// ---- TMA bulk copy + mbarrier  ---------------------------------------------------------
__device__ __forceinline__ uint32_t smem_u32(const void* p) { return (uint32_t)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void mbar_init(unsigned long long* b, int count) {
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(b)), "r"(count) : "memory");
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
}
__device__ __forceinline__ void mbar_expect_tx(unsigned long long* b, uint32_t bytes) {
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(b)), "r"(bytes) : "memory");
}
__device__ __forceinline__ void bulk_g2s(void* dst, const void* src, uint32_t bytes, unsigned long long* b) {
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];" ::"r"(smem_u32(dst)),
                 "l"(src), "r"(bytes), "r"(smem_u32(b))
                 : "memory");
}
__device__ __forceinline__ void mbar_wait(unsigned long long* b, uint32_t parity) {
    uint32_t ok;
    do {
        asm volatile("{\n .reg .pred p;\n mbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n selp.u32 %0, 1, 0, p;\n}"
                     : "=r"(ok)
                     : "r"(smem_u32(b)), "r"(parity)
                     : "memory");
    } while (!ok);
}

// ---- small reductions ---------------------------------------------------------------------------------
__device__ __forceinline__ double warp_sum(double v) {
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
    return v;
}

// Block-wide sums of NV doubles; result valid in all threads.  `scratch` holds NV * (NT/32) doubles.
template <int NT, int NV>
__device__ __forceinline__ void block_sum(double (&v)[NV], double* scratch) {
    constexpr int NW = NT / 32;
    int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
#pragma unroll
    for (int i = 0; i < NV; ++i) v[i] = warp_sum(v[i]);
    __syncthreads();  // protect scratch from a previous use
    if (lane == 0)
#pragma unroll
        for (int i = 0; i < NV; ++i) scratch[i * NW + wid] = v[i];
    __syncthreads();
#pragma unroll
    for (int i = 0; i < NV; ++i) {
        double s = 0.0;
#pragma unroll
        for (int k = 0; k < NW; ++k) s += scratch[i * NW + k];
        v[i] = s;
    }
}

// ---- kernel parameter blocks --------------------------------------------------------------------------
struct EventSetDev {
    int32_t n_events;
    int32_t max_ns, max_nz;
    const int64_t* sample_off;  // [n_events+1]
    const int64_t* grid_off;    // [n_events+1]
    const float4* rec;          // packed sample records {A, B} (see above), sorted by d_L within each event
    const int32_t* perm;        // sorted position -> caller's index within the event
    const double* zc;           // z_g - z0_i  (centred grid)
    const float* qn;            // p_gal(z_g) * trapezoid weight / (the event's largest such product)
    const double* uni_dz;       // [n_events] grid spacing if the event's grid is equally spaced, else 0
    const double* max_dz;       // [n_events] largest grid spacing of the event
    const double* z0;           // [n_events] centre of each event's grid
    const double* lnm1_lo;      // [n_events] smallest / largest ln m1d of the event's samples
    const double* lnm1_hi;
    const float2* chunk_top;    // [n_events][kFastWarps] k_events_fast: {largest m2d, t of the last sample} of every warp's chunk
                                // (laid out for the warps of the event's class: fast_warps_for(N_s))
    const int32_t* k_lo;        // [n_events] first / last row of the z(ln d_L) table the event's samples address
    const int32_t* k_hi;
    const double* fixed_bw;     // [n_events] or null
    // Epanechnikov kernel: prefix sums over the event grid (N_z + 1 entries per event, offset grid_off[i] + i) of
    // q_g, q_g z'_g, q_g z'_g^2 (z' = z_g - z0, q as in qn but fp64)
    const double* ep_q0; const double* ep_q1; const double* ep_q2;
    // event-local polynomials (k_events, S2): centre and half-width of the event's samples in table coordinates
    // (tk_h = 0: the event's d_L range is too wide for them), and the same centre / scale for the 12.20 fixed point
    const double* tk_c;         // [n_events]
    const double* tk_h;         // [n_events]
    const int64_t* poly_off;    // [n_events+1] offsets into prec (events padded to a multiple of 32 samples)
    const float4* prec_a;       // records of the polynomial sweep: {m1d, m2d, t in [-1,1], ln m1d}
    const float2* prec_b;       //                                  {ln m2d, log2(1/prior) - scale}
    // k_events_fast: qn again with every event's slice starting at a multiple of 4 floats and zero-padded to one (TMA source)
    const float* qn4;
    const int64_t* q4_off;      // [n_events]
};

struct EventKernelParams {
    EventSetDev ev;
    const LamConst* Lc;      // [n_lambda]
    const Row* tab;          // [n_lambda][rows]
    const MassRow* mtab;     // [n_lambda][2][n_mass+2]
    const double* dc_tab;    // [n_lambda][n_table+1+kZPad] (placement ON_GRID only) or null
    int32_t n_lambda, tab_rows, n_mass, n_table;
    int32_t placement, bw_rule, kde_method, kde_kernel, n_bins;
    float neff_min;          // below this Kish n_eff the fp32 polynomial sweep is redone by the careful one
    double z_table_max, cutoff;
    double* logI;            // [n_lambda][n_events]
    uint32_t* flags;         // [n_lambda]
    unsigned long long* stats;  // [0] executed pairs (incl. band padding), [1] pairs inside the cut-off
    const double* ln_shift;  // [n_events] prior scale factored out of the weights, added back to log I
    const double* ln_qscale; // [n_events] ln of the event's largest q_g (qn = q / that), added back to log I
    const float* poly;       // [n_lambda][n_events][4 kPolyN] event-local polynomials fitted by k_polyfit
    const int32_t* ev_list;  // null, or the events this launch covers (n_ev_list of them; the others belong to k_events_fast)
    int32_t n_ev_list;
    const uint32_t* worklist;      // null, or the units (lambda * n_events + event) handed over by k_events_fast ...
    const unsigned int* work_count;// ... and their number; worklist_ctas CTAs loop over them
    int32_t worklist_ctas;
    // diagnostics (single event, single lambda) -- null in the hot path
    int32_t dbg_event;       // >= 0: blockIdx.x addresses lambda only, event = dbg_event
    double* dbg_z; double* dbg_w; double* dbg_h; double* dbg_K;
};

// k_events_fast (k_events_fast.cu): the regular units; everything else goes to k_events through the work list
struct FastEventParams {
    EventSetDev ev;
    const LamConst* Lc;
    const MassRow* mtab;     // [n_lambda][2][n_mass+2]
    const float* poly;       // [n_lambda][n_events][4 kPolyN]
    int32_t n_lambda, n_mass, bw_rule;
    float neff_min;          // units with a Kish n_eff below this are handed over (k_events takes its careful sweep there)
    double cutoff;
    double* logI;            // [n_lambda][n_events]
    const double* ln_shift; const double* ln_qscale;
    const int32_t* fast_events;   // the events this launch takes (narrow d_L range, equally spaced grid; one class)
    int32_t warps, max_d, max_ns; // the class: warps per CTA, psi-table cap, longest sample list (sizes the shared memory)
    uint32_t* worklist; unsigned int* work_count;
};

struct InjSetDev {
    int64_t n_det;
    double n_inj_total;
    const float4* rec;       // packed injection records {A, B}, sorted by d_L
    const int64_t* perm;
    // chunk-local polynomials (k_inject): records {m1d, m2d, t, ln m1d}, {ln m2d, log2(1/p_draw) - scale} padded to
    // whole chunks, centre / half-width of each chunk in table coordinates (tk_h = 0: range too wide -> table path)
    const float4* prec_a;
    const float2* prec_b;
    const double* tk_c;      // [n_chunks]
    const double* tk_h;      // [n_chunks]
    const float* blk_m2d;    // [n_chunks][64] largest m2d of every block of 256 injections (chunks are ordered by m2d)
};

struct InjKernelParams {
    InjSetDev inj;
    const LamConst* Lc; const Row* tab; const MassRow* mtab;
    int32_t n_lambda, tab_rows, n_mass, chunk;  // chunk = injections per block
    double z_table_max, z_cat_max;
    double2* partial;        // [n_blocks][n_lambda] {sum s, sum s^2}
    uint32_t* flags;
    const float* poly;       // [n_lambda][n_chunks][4 kPolyN] chunk-local polynomials fitted by k_polyfit
    int32_t n_chunks;
    double* dbg_s;           // diagnostics: per-injection s_j (caller order), single lambda
    double dbg_scale;        // exp(ln_shift) to undo the draw-density scale in dbg_s
};

struct CombineParams {
    const LamConst* Lc; const double* logI; const double2* partial;
    int32_t n_lambda, n_events, n_inj_blocks;
    int64_t n_det; double n_inj_total, neff_factor;
    double inj_ln_shift;     // draw-density scale factored out of s_j, added back to log xi
    int32_t n_groups;        // many-1d: > 0 = physical events, each the sub-events [group_off[g], group_off[g+1])
    const int64_t* group_off; const double* ln_factor;
    const uint32_t* flags_in;
    double* out_loglike; double* out_event_logI; double* out_logxi; double* out_neff; uint32_t* out_flags;
};

// host-callable launchers (defined in the .cu files)
cudaError_t launch_tables(const double* lam, int n_lambda, const TableParams& P, LamConst* Lc, double* dc_tab,
                          Row* tab_ev, Row* tab_inj, MassRow* mtab, cudaStream_t st);

cudaError_t launch_polyfit(const LamConst* Lc, const Row* tab, int tab_rows, int n_lambda, int n_ranges, const double* tk_c,
                           const double* tk_h, const double* z_ref, double z_ref_const, bool is_inj, const double* pm,
                           const double* lnm1_lo, const double* lnm1_hi, int n_mass, int mcap, double dx_tab, float* out, cudaStream_t st);
int events_mass_stage_rows(int n_mass);   // rows of the mass table a k_events CTA stages per variant
cudaError_t launch_events(const EventKernelParams& P, bool count_pairs, cudaStream_t st);
cudaError_t launch_events_fast(const FastEventParams& P, int n_fast, cudaStream_t st);
size_t events_fast_smem_bytes(int max_ns, int max_nz, int warps, int max_d);
cudaError_t launch_inject(const InjKernelParams& P, int n_blocks, cudaStream_t st);
cudaError_t launch_combine(const CombineParams& P, cudaStream_t st);
cudaError_t launch_table_lookup(const LamConst* Lc, const Row* tab, DlGrid g, int64_t n, const double* dL,
                                double z_table_max, double* z_out, double* r_out, cudaStream_t st);
cudaError_t launch_pcat(double Om, int n_los, const int64_t* gal_off, const double* zt, const double* st, const double* wg,
                        const int64_t* grid_off, const double* zg, double* coef, double* out, cudaStream_t st_);
// (k_pcat_static.cu) k_pcat with its per-galaxy scratch in a file-scope __device__ array: no allocation anywhere
cudaError_t launch_pcat_static(double Om, int n_los, long long n_gal, const int64_t* gal_off, const double* zt, const double* st,
                               const double* wg, const int64_t* grid_off, const double* zg, double* out, cudaStream_t st_);
int pcat_static_max_galaxies();
cudaError_t launch_pgal(double Om, double zmax, int n_los, const int64_t* compl_off, const double* zc, const double* pc,
                        const int64_t* grid_off, const double* zg, double* out, double* fr_out, cudaStream_t st_);
cudaError_t launch_grad_expand(const double* lam, int n_lambda, double rel, double* ext, cudaStream_t st);
cudaError_t launch_grad_combine(const double* lam, int n_lambda, double rel, const double* ll, const uint32_t* fl, double* out_ll,
                                double* out_grad, uint32_t* out_fl, cudaStream_t st);
int grad_rows();
cudaError_t upload_gauss_legendre();   // fills the __constant__ node tables used by S1
cudaError_t measure_alu_peaks(int n_sm, int reps, cudaStream_t st, double out_g[4]);
size_t events_smem_bytes(int max_ns, int max_nz);
size_t tables_smem_bytes(const TableParams& P);
size_t inject_smem_bytes(int n_mass);

}  // namespace chim
