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
    uint32_t flags;     // CHIM_FLAG_LAMBDA_DOMAIN | CHIM_FLAG_DL_NONMONOTONE
    int32_t beta_is_m1; // |beta + 1| < 1e-12 : log form of the power integral
};

// One interval of the per-lambda interpolation table in x = ln d_L: cubic (Lagrange through 4 nodes,
// expanded in the local coordinate t in [0,1)) for 4 columns:
//   0: z      1: u = ln(1+z)      2: a = 1/(1+z)      3: R = smooth redshift factor of the weight
// (events: psi/J or 1; injections: psi u_vol / J).  128 B = one cache line.
struct __align__(16) Row {
    double c[4][4];  // c[col][degree]
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

// One interval of the per-lambda mass table in y = ln m1: cubics (local coordinate t in [0,1)) of
//   a: ln[ p(m1)/S(m1) * m1'^2 S(m1)/C(m1) ]  with the power law present (m1 <= m_high),  m1' = m1 - m_low
//   b: the same with the Gaussian component only (m1 > m_high)
// i.e. ln of  p(m1) / C(m1) * m1'^2  -- smooth and finite on [m_low, inf) because C/S ~ rho m1'^2 (M3/M4).
struct __align__(16) MassRow {
    double a[4], b[4];
};

// exp(x) for the sample kernels: fp64 range reduction x log2(e) = n + f, |f| <= 1/2 (exact in fp64), MUFU.EX2 on
// the fp32 remainder (relative error <= 2.4e-7), 2^n through the exponent field.  |x| must stay
// below ~1e9 (the magic-number rounding) -- every caller bounds its argument; n is clamped so that the result never
// leaves the normal range: e^-707 ~ 1e-307 stands in for 0.
__device__ __forceinline__ double exp_mufu(double x) {
    const double y = x * 1.4426950408889634074;
    const double t = y + 6755399441055744.0;            // 1.5 * 2^52: round to nearest integer
    int n = __double2loint(t);
    const double fn = t - 6755399441055744.0;
    const float f = (float)(y - fn);
    float e;
    asm("ex2.approx.ftz.f32 %0, %1;" : "=f"(e) : "f"(f));
    n = max(-1020, min(n, 1020));
    const double ed = (double)e;                        // in [0.70, 1.42]
    return __hiloint2double(__double2hiint(ed) + (n << 20), __double2loint(ed));
}

// 1/x for finite non-zero normal x: MUFU.RCP64H seed + two Newton steps (error ~1e-16), no special cases.
__device__ __forceinline__ double fast_rcp(double x) {
    double r;
    asm("rcp.approx.ftz.f64 %0, %1;" : "=d"(r) : "d"(x));
    double e = fma(-x, r, 1.0);
    r = fma(r, e, r);
    e = fma(-x, r, 1.0);
    return fma(r, e, r);
}

__device__ __forceinline__ double horner3(const double* c, double t) {
    return fma(fma(fma(c[3], t, c[2]), t, c[1]), t, c[0]);
}

// Where a thread finds the per-lambda mass table: rows [lo, lo + cap) of the "a" variant staged in shared memory as
// two split arrays (16-byte halves: the layout with the fewest bank conflicts for scattered rows), everything else
// (rows outside the staged range, the Gaussian-only "b" variant beyond m_high) in global memory.
struct MassLookup {
    const MassRow* g;          // [n_mass + 2] rows of this lambda
    const double2* sA;         // staged {a[0], a[1]} or null
    const double2* sB;         // staged {a[2], a[3]}
    int lo, cap, n_mass;
};

// Streaming 128-bit read of a packed sample record: read once per CTA, so it must not evict the table rows from L1.
__device__ __forceinline__ double2 ldg_stream(const double2* p) {
    double2 v;
    asm volatile("ld.global.nc.L1::no_allocate.v2.f64 {%0,%1}, [%2];" : "=d"(v.x), "=d"(v.y) : "l"(p));
    return v;
}
__device__ __forceinline__ void prefetch_l1(const void* p) { asm volatile("prefetch.global.L1 [%0];" ::"l"(p)); }

__device__ __forceinline__ double2 ldg256_lo(const double* p, double2& hi) {   // one 256-bit read-only load
    double2 lo;
    asm("ld.global.nc.v4.f64 {%0,%1,%2,%3}, [%4];" : "=d"(lo.x), "=d"(lo.y), "=d"(hi.x), "=d"(hi.y) : "l"(p));
    return lo;
}

// Steps S2 / S5 for one sample (or injection): redshift from the table, source-frame masses, population weight
//   w = p(m1, m2 | lambda_m) * R(z) / prior,   p(m1,m2) = p(m1) m2^beta S(m2) / C(m1)     (M1-M4)
// assembled in log space from two table look-ups:
//   ln w' = LQ(ln m1) + beta ln m2 + ln R + ln(1/prior),   w = exp(ln w') S(m2) / m1'^2
//   LQ   per-lambda mass table (MassRow): ln[p(m1)/C(m1) m1'^2], smooth on [m_low, inf)
//   S(m2) = 1/(1 + exp(delta/m2' + delta/(m2' - delta))) inside the window, 1 above (M1)
//   ln R, z, ln(1+z), 1/(1+z): the four cubics of the sample's row of the z(ln d_L) table
//   PAPER.md:52 (d_L -> z, m = m^d/(1+z)), :195-198 eq. 20 (mass model), :226 eq. 21, :75 eq. 11.
// Two exponentials (MUFU.EX2 on fp64-reduced arguments) and two reciprocals per sample; selects instead of
// data-dependent branches, except the (rare) fall-back of the mass row to global memory.
__device__ __forceinline__ void sample_weight(const LamConst& L, const Row* __restrict__ tab, int n_rows,
                                              const MassLookup& M, double tkmax, double z_table_max,
                                              double tk, double m1d, double q, double lnm1d, double lnq, double lnipr,
                                              double& z, double& w, bool& out_of_range) {
    out_of_range = !(tk <= tkmax);
    int k = (int)((tk < (double)(n_rows - 2)) ? tk : (double)(n_rows - 2));
    k = max(1, k);
    double t = tk - (double)k;
    const double* rp = reinterpret_cast<const double*>(tab + k);     // 4 x 256-bit loads of one 128-byte row
    double2 c0, c1, c2, c3, c4, c5, c6, c7;
    c0 = ldg256_lo(rp, c1);
    c2 = ldg256_lo(rp + 4, c3);
    c4 = ldg256_lo(rp + 8, c5);
    c6 = ldg256_lo(rp + 12, c7);
    double zt = fma(fma(fma(c1.y, t, c1.x), t, c0.y), t, c0.x);
    double u = fma(fma(fma(c3.y, t, c3.x), t, c2.y), t, c2.x);
    double a = fma(fma(fma(c5.y, t, c5.x), t, c4.y), t, c4.x);
    double lnR = fma(fma(fma(c7.y, t, c7.x), t, c6.y), t, c6.x);
    z = out_of_range ? z_table_max : zt;
    const double m1 = m1d * a, m2 = q * m1;
    const double lm1 = lnm1d - u, lm2 = lm1 + lnq;
    const double mp1 = m1 - L.m_low, mp2 = m2 - L.m_low;
    // mass table
    double tm = fma(lm1 - L.lm0, L.inv_dlm, 1.0);
    int km = max(1, min((int)tm, M.n_mass));
    tm -= (double)km;
    double2 d0, d1;
    const int ks = km - M.lo;
    if ((unsigned)ks < (unsigned)M.cap && m1 <= L.m_high) {
        d0 = M.sA[ks];
        d1 = M.sB[ks];
    } else {
        d0 = ldg256_lo(reinterpret_cast<const double*>(M.g + km) + ((m1 <= L.m_high) ? 0 : 4), d1);
    }
    double lnw = fma(fma(fma(d1.y, tm, d1.x), tm, d0.y), tm, d0.x);
    lnw += fma(L.beta, lm2, lnR + lnipr);
    // smoothing of m2 (M1): f = delta (2 m' - delta) / (m' (m' - delta)), m' clamped strictly inside the window
    const double lo = L.delta * 1e-3, hi = L.delta * (1.0 - 1e-12);   // S(m' < 1e-3 delta) < e^-998: "0" either way
    double mc = (mp2 > lo) ? mp2 : lo;
    mc = (mc < hi) ? mc : hi;
    const double f = L.delta * (2.0 * mc - L.delta) * fast_rcp(mc * (mc - L.delta));
    const double S2 = fast_rcp(1.0 + exp_mufu(f));
    const double r1 = fast_rcp((mp1 > 0.0) ? mp1 : 1.0);
    double v = exp_mufu(lnw) * (r1 * r1);
    v = (mp2 < L.delta) ? v * S2 : v;
    const bool ok = !out_of_range && (mp2 > 0.0);      // R15 support: m_low < m2 (<= m1)
    w = ok ? v : 0.0;
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
    const double2* recA;        // {tk, m1d}         per sample, sorted by d_L within each event
    const double2* recB;        // {q = m2d/m1d, ln m1d}
    const double2* recC;        // {ln q, 1/pi}
    const int32_t* perm;        // sorted position -> caller's index within the event
    const double* zc;           // z_g - z0_i  (centred grid)
    const float* qn;            // p_gal(z_g) * trapezoid weight / (the event's largest such product)
    const double* uni_dz;       // [n_events] grid spacing if the event's grid is equally spaced, else 0
    const double* z0;           // [n_events] centre of each event's grid
    const double* lnm1_lo;      // [n_events] smallest / largest ln m1d of the event's samples
    const double* lnm1_hi;
    const double* fixed_bw;     // [n_events] or null
};

struct EventKernelParams {
    EventSetDev ev;
    const LamConst* Lc;      // [n_lambda]
    const Row* tab;          // [n_lambda][rows]
    const MassRow* mtab;     // [n_lambda][n_mass+2]
    const double* dc_tab;    // [n_lambda][n_table+1+kZPad] (placement ON_GRID only) or null
    int32_t n_lambda, tab_rows, n_mass, n_table;
    int32_t placement, bw_rule, kde_method;
    double z_table_max, cutoff;
    double* logI;            // [n_lambda][n_events]
    uint32_t* flags;         // [n_lambda]
    unsigned long long* stats;  // [0] executed pairs (incl. band padding), [1] pairs inside the cut-off
    const double* ln_shift;  // [n_events] prior scale factored out of the weights, added back to log I
    const double* ln_qscale; // [n_events] ln of the event's largest q_g (qn = q / that), added back to log I
    // diagnostics (single event, single lambda) -- null in the hot path
    int32_t dbg_event;       // >= 0: blockIdx.x addresses lambda only, event = dbg_event
    double* dbg_z; double* dbg_w; double* dbg_h; double* dbg_K;
};

struct InjSetDev {
    int64_t n_det;
    double n_inj_total;
    const double2* recA; const double2* recB; const double2* recC;  // sorted by d_L
    const int64_t* perm;
};

struct InjKernelParams {
    InjSetDev inj;
    const LamConst* Lc; const Row* tab; const MassRow* mtab;
    int32_t n_lambda, tab_rows, n_mass, chunk;  // chunk = injections per block
    double z_table_max, z_cat_max;
    double2* partial;        // [n_blocks][n_lambda] {sum s, sum s^2}
    uint32_t* flags;
    double* dbg_s;           // diagnostics: per-injection s_j (caller order), single lambda
    double dbg_scale;        // exp(ln_shift) to undo the draw-density scale in dbg_s
};

struct CombineParams {
    const LamConst* Lc; const double* logI; const double2* partial;
    int32_t n_lambda, n_events, n_inj_blocks;
    int64_t n_det; double n_inj_total, neff_factor;
    double inj_ln_shift;     // draw-density scale factored out of s_j, added back to log xi
    const uint32_t* flags_in;
    double* out_loglike; double* out_event_logI; double* out_logxi; double* out_neff; uint32_t* out_flags;
};

// host-callable launchers (defined in the .cu files)
cudaError_t launch_tables(const double* lam, int n_lambda, const TableParams& P, LamConst* Lc, double* dc_tab,
                          Row* tab_ev, Row* tab_inj, MassRow* mtab, cudaStream_t st);

cudaError_t launch_events(const EventKernelParams& P, cudaStream_t st);
cudaError_t launch_inject(const InjKernelParams& P, int n_blocks, cudaStream_t st);
cudaError_t launch_combine(const CombineParams& P, cudaStream_t st);
cudaError_t launch_table_lookup(const LamConst* Lc, const Row* tab, DlGrid g, int64_t n, const double* dL,
                                double z_table_max, double* z_out, double* r_out, cudaStream_t st);
cudaError_t upload_gauss_legendre();   // fills the __constant__ node tables used by S1
cudaError_t measure_alu_peaks(int n_sm, int reps, cudaStream_t st, double out_g[4]);
size_t events_smem_bytes(int max_ns, int max_nz);
size_t tables_smem_bytes(const TableParams& P);
size_t inject_smem_bytes(int n_mass);

}  // namespace chim
