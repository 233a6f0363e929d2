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
    DlGrid ev, inj;
};

// exp(x) in fp64 for the sample kernels: argument clamped to [-700, 700] (e^-700 ~ 1e-304 stands in for 0,
// nothing on this path needs more), Cody-Waite reduction x = n ln2 + r with |r| <= ln2/2, degree-11 Taylor
// polynomial in Horner form (relative error < 1e-14), scaling by 2^n through the exponent field.  Branch-free;
// the coefficients live in constant memory so that DFMA takes them as direct operands.
static __constant__ double c_exp_coef[12] = {
    2.50521083854417187751e-08, 2.75573192239858906526e-07, 2.75573192239858906526e-06, 2.48015873015873015873e-05,
    1.98412698412698412698e-04, 1.38888888888888888889e-03, 8.33333333333333333333e-03, 4.16666666666666666667e-02,
    1.66666666666666666667e-01, 0.5, 1.0, 1.0};
static __constant__ double c_exp_red[5] = {1.4426950408889634074, 6755399441055744.0 /* 1.5 * 2^52 */,
                                           -6.93147180369123816490e-01, -1.90821492927058770002e-10, 700.0};

__device__ __forceinline__ double fast_exp(double x) {
    x = (x > -c_exp_red[4]) ? x : -c_exp_red[4];       // cheap clamps (no NaN canonicalisation): inputs are finite
    x = (x < c_exp_red[4]) ? x : c_exp_red[4];
    double t = fma(x, c_exp_red[0], c_exp_red[1]);     // round-to-nearest integer by the magic-number addition
    int n = __double2loint(t);
    double fn = t - c_exp_red[1];
    double r = fma(fn, c_exp_red[2], x);
    r = fma(fn, c_exp_red[3], r);
    double p = c_exp_coef[0];
#pragma unroll
    for (int i = 1; i < 12; ++i) p = fma(p, r, c_exp_coef[i]);
    return p * __hiloint2double((n + 1023) << 20, 0);  // |n| <= 1010: 2^n is a normal double
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

// Smoothing denominator 1/S(m) = 1 + exp(f(m')), f = delta/m' + delta/(m'-delta) = delta (2m'-delta)/(m'(m'-delta))
// (M1), for m' = m - m_low clamped strictly inside the window so that the expression is finite for every lane
// (lanes outside the window discard the value).
__device__ __forceinline__ double smooth_den(double mp, const LamConst& L) {
    const double lo = L.delta * 1e-6, hi = L.delta * (1.0 - 1e-12);
    double mpc = (mp > lo) ? mp : lo;
    mpc = (mpc < hi) ? mpc : hi;
    double f = L.delta * (2.0 * mpc - L.delta) * fast_rcp(mpc * (mpc - L.delta));
    return 1.0 + fast_exp(f);
}

// Inside the window both S(m1) and C(m1) = int_{m_low}^{m1} m^beta S(m) dm (M3/M4) vanish faster than any power
// at m_low, so the table holds the smooth ratio rho(m') = C / (S m'^2) (rho -> m_low^beta/delta_m as m' -> 0,
// rho(delta_m) = W_c/delta_m^2): S(m1)/C(m1) = 1/(rho m'^2) and S(m1) cancels analytically in the weight.
// Cubic Lagrange on uniform nodes.
__device__ __forceinline__ double rho_window(double mp, const LamConst& L, const double* __restrict__ rtab, int n_win) {
    double x = mp * L.win_scale;
    int b = (int)x - 1;
    b = max(0, min(b, n_win - 3));
    double s = x - (double)b;   // in [0, 3]
    double s1 = s - 1.0, s2 = s - 2.0, s3 = s - 3.0;
    double l0 = -s1 * s2 * s3 * (1.0 / 6.0), l1 = s * s2 * s3 * 0.5, l2 = -s * s1 * s3 * 0.5, l3 = s * s1 * s2 * (1.0 / 6.0);
    return l0 * rtab[b] + l1 * rtab[b + 1] + l2 * rtab[b + 2] + l3 * rtab[b + 3];
}

// Steps S2 / S5 for one sample (or injection): redshift from the table, source-frame masses, population
// weight.  `ipr` = 1/pi_j (events) or 1/p_draw,j (injections); R carries psi/J (and u_vol for injections).
//   PAPER.md:52 (d_L -> z, m = m^d/(1+z)), :195-198 eq. 20 + M1-M4 (mass model), :226 eq. 21, :75 eq. 11.
// Written without data-dependent branches (selects only): the lanes of a warp hold samples on both sides of
// every mass-function edge, so branches would serialise the exponentials.
__device__ __forceinline__ void sample_weight(const LamConst& L, const Row* __restrict__ tab, int n_rows,
                                              const double* __restrict__ wtab, int n_win, double tkmax,
                                              double z_table_max, double tk, double m1d, double q, double lnm1d,
                                              double lnq, double ipr, double& z, double& w, bool& out_of_range) {
    out_of_range = !(tk <= tkmax);
    int k = (int)((tk < (double)(n_rows - 2)) ? tk : (double)(n_rows - 2));
    k = max(1, k);
    double t = tk - (double)k;
    const double2* rp = reinterpret_cast<const double2*>(tab + k);   // 8 x 128-bit loads of one 128-byte row
    double2 c0 = rp[0], c1 = rp[1], c2 = rp[2], c3 = rp[3], c4 = rp[4], c5 = rp[5], c6 = rp[6], c7 = rp[7];
    double zt = fma(fma(fma(c1.y, t, c1.x), t, c0.y), t, c0.x);
    double u = fma(fma(fma(c3.y, t, c3.x), t, c2.y), t, c2.x);
    double a = fma(fma(fma(c5.y, t, c5.x), t, c4.y), t, c4.x);
    double R = fma(fma(fma(c7.y, t, c7.x), t, c6.y), t, c6.x);
    z = out_of_range ? z_table_max : zt;
    double m1 = m1d * a, m2 = q * m1;
    double lm1 = lnm1d - u, lm2 = lm1 + lnq;
    double bl2 = L.beta * lm2;                                      // ln m2^beta
    double dm = m1 - L.mu;
    double e = fast_exp(L.a_g - dm * dm * L.inv2s2 + bl2);          // lambda_g N(m1) m2^beta / Z1
    double epl = fast_exp(L.a_pl - L.alpha * lm1 + bl2);            // (1-lambda_g) PL(m1) m2^beta / Z1
    e += (m1 <= L.m_high) ? epl : 0.0;
    double mp1 = m1 - L.m_low, mp2 = m2 - L.m_low;
    double den2 = smooth_den(mp2, L);
    double den = (mp2 < L.delta) ? den2 : 1.0;                      // 1/S(m2)
    // C(m1): above the window W_c + closed-form power integral; inside, rho m'^2 (S(m1) cancelled)
    double pw = L.beta_is_m1 ? (lm1 - L.ln_mc) : (fast_exp(L.bp1 * lm1) - L.pow_mc_bp1) * L.inv_bp1;
    double mp1c = (mp1 > 0.0) ? mp1 : 0.0;
    mp1c = (mp1c < L.delta) ? mp1c : L.delta;
    double cw = rho_window(mp1c, L, wtab, n_win) * mp1c * mp1c;
    double C = (mp1 < L.delta) ? cw : L.W_c + pw;
    double dc = den * C;
    bool ok = !out_of_range && (m2 >= L.m_low) && (dc > 1e-300) && (dc < 1e300);   // R15 support; underflowed S or C
    w = ok ? e * R * ipr * fast_rcp(ok ? dc : 1.0) : 0.0;
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
    const double* qg;           // p_gal(z_g) * trapezoid weight
    const double* z0;           // [n_events] centre of each event's grid
    const double* fixed_bw;     // [n_events] or null
};

struct EventKernelParams {
    EventSetDev ev;
    const LamConst* Lc;      // [n_lambda]
    const Row* tab;          // [n_lambda][rows]
    const double* wtab;      // [n_lambda][n_win+1]  rho(m') nodes
    const double* dc_tab;    // [n_lambda][n_table+1+kZPad] (placement ON_GRID only) or null
    int32_t n_lambda, tab_rows, n_win, n_table;
    int32_t placement, bw_rule;
    double z_table_max, cutoff;
    double* logI;            // [n_lambda][n_events]
    uint32_t* flags;         // [n_lambda]
    unsigned long long* stats;  // [0] evaluated pairs
    const double* ln_shift;  // [n_events] prior scale factored out of the weights, added back to log I
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
    const LamConst* Lc; const Row* tab; const double* wtab;
    int32_t n_lambda, tab_rows, n_win, chunk;  // chunk = injections per block
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
                          Row* tab_ev, Row* tab_inj, double* wtab, cudaStream_t st);
cudaError_t launch_events(const EventKernelParams& P, cudaStream_t st);
cudaError_t launch_inject(const InjKernelParams& P, int n_blocks, cudaStream_t st);
cudaError_t launch_combine(const CombineParams& P, cudaStream_t st);
cudaError_t launch_table_lookup(const LamConst* Lc, const Row* tab, DlGrid g, int64_t n, const double* dL,
                                double z_table_max, double* z_out, double* r_out, cudaStream_t st);
cudaError_t upload_gauss_legendre();   // fills the __constant__ node tables used by S1
cudaError_t measure_alu_peaks(int n_sm, int reps, cudaStream_t st, double out_g[4]);
size_t events_smem_bytes(int max_ns, int max_nz);
size_t tables_smem_bytes(const TableParams& P);

}  // namespace chim
