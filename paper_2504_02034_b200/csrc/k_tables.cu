// k_tables.cu -- step S1: per-lambda table builder (one CTA per lambda).
//
//   d_C(z) = (c/H0) int_0^z dz'/E(z'),  E = sqrt(Om (1+z)^3 + 1 - Om)      (eq. 1, R4)
//       cumulative trapezoid of 1/E on a uniform z grid + the Euler-Maclaurin end term
//       (f'_k - f'_{k+1}) dz^2/12 per panel (f' analytic), block-wide prefix sum in fp64;
//   d_L^gw(z) = Xi(z) (1+z) d_C(z),  Xi = Xi0 + (1-Xi0)/(1+z)^n               (eq. 2)
//       with the monotonicity check of R16 at the table nodes;
//   z(ln d_L) tables: for each node of a uniform grid in x = ln d_L the redshift is found by bisection
//       over the d_L^gw nodes and Newton on the cubic-Hermite d_C (node slopes c/H exact); the nodes of
//       z, ln(1+z), 1/(1+z) and the smooth weight factor psi/J (PAPER.md:226 eq. 21, :75 eq. 11) are turned
//       into per-interval cubic coefficients so that the sample kernels do one Horner evaluation per
//       column (the sample's table coordinate is lambda-independent and precomputed at init);
//   mass function (M1-M4): N_pl, Z1 (32-node Gauss-Legendre on the smoothing window + closed-form tails), the
//       cumulative window integral W(m) = int_{m_low}^m m'^beta S(m') dm', and from them the per-lambda mass table
//       LQ(ln m1) = ln[ p(m1)/C(m1) * (m1 - m_low)^2 ] (two variants: with / without the power law, for m1 on
//       either side of m_high) as per-interval cubics -- the sample kernels then need one exponential per sample.
#include "chim_internal.cuh"

namespace chim {

__constant__ double c_glw_x[kGLWin], c_glw_w[kGLWin];      // GL nodes/weights on [-1,1]
__constant__ double c_glp_x[kGLPanel], c_glp_w[kGLPanel];

// Host: Gauss-Legendre rule by Newton iteration on the three-term recurrence, symmetric fill.
static void gauss_legendre_host(int n, double* x, double* w) {
    const double pi = 3.14159265358979323846;
    for (int i = 0; i < (n + 1) / 2; ++i) {
        double t = cos(pi * (4 * i + 3) / (4.0 * n + 2.0));
        double pn = 0.0, dpn = 1.0;
        for (int it = 0; it < 64; ++it) {
            double pkm1 = 1.0, pk = t;
            for (int k = 1; k < n; ++k) {
                double pkp1 = ((2 * k + 1) * t * pk - k * pkm1) / (k + 1);
                pkm1 = pk;
                pk = pkp1;
            }
            pn = pk;
            dpn = n * (pkm1 - t * pk) / (1.0 - t * t);
            double dt = pn / dpn;
            t -= dt;
            if (fabs(dt) < 1e-16) break;
        }
        // re-evaluate the derivative at the converged root
        double pkm1 = 1.0, pk = t;
        for (int k = 1; k < n; ++k) {
            double pkp1 = ((2 * k + 1) * t * pk - k * pkm1) / (k + 1);
            pkm1 = pk;
            pk = pkp1;
        }
        dpn = n * (pkm1 - t * pk) / (1.0 - t * t);
        x[i] = -t;
        x[n - 1 - i] = t;
        w[i] = w[n - 1 - i] = 2.0 / ((1.0 - t * t) * dpn * dpn);
    }
}

cudaError_t upload_gauss_legendre() {
    double x[kGLWin], w[kGLWin];
    gauss_legendre_host(kGLWin, x, w);
    cudaError_t e = cudaMemcpyToSymbol(c_glw_x, x, sizeof(double) * kGLWin);
    if (e != cudaSuccess) return e;
    e = cudaMemcpyToSymbol(c_glw_w, w, sizeof(double) * kGLWin);
    if (e != cudaSuccess) return e;
    gauss_legendre_host(kGLPanel, x, w);
    e = cudaMemcpyToSymbol(c_glp_x, x, sizeof(double) * kGLPanel);
    if (e != cudaSuccess) return e;
    return cudaMemcpyToSymbol(c_glp_w, w, sizeof(double) * kGLPanel);
}

constexpr int kTabThreads = 256;

struct TabSmem {
    LamConst L;
    double red[4 * (kTabThreads / 32)];
    double scan[kTabThreads];
    int ibad;
};

__device__ __forceinline__ double invE(double z, double Om) {
    double a = 1.0 + z;
    return rsqrt(Om * a * a * a + 1.0 - Om);
}
// d(1/E)/dz = -3 Om (1+z)^2 / (2 E^3)
__device__ __forceinline__ double dinvE(double z, double Om) {
    double a = 1.0 + z;
    double ie = rsqrt(Om * a * a * a + 1.0 - Om);
    return -1.5 * Om * a * a * ie * ie * ie;
}
__device__ __forceinline__ double Xi_of(double z, const LamConst& L) { return L.Xi0 + (1.0 - L.Xi0) * exp(-L.n * log1p(z)); }
__device__ __forceinline__ double dXi_of(double z, const LamConst& L) {
    return -L.n * (1.0 - L.Xi0) * exp(-(L.n + 1.0) * log1p(z));
}
// Madau-Dickinson rate, eq. (21) with constant 1 (R5), from u = ln(1+z)
__device__ __forceinline__ double psi_of_u(double u, const LamConst& L) {
    return exp(L.gamma * u) / (1.0 + exp(L.gk * (u - L.ln1pzp)));
}
__device__ __forceinline__ double smooth_S_dev(double m, const LamConst& L) {
    if (m <= L.m_low) return 0.0;
    if (m >= L.m_c) return 1.0;
    double mp = m - L.m_low;
    double f = L.delta / mp + L.delta / (mp - L.delta);
    return 1.0 / (1.0 + exp(f));
}
__device__ __forceinline__ double powerlaw_unnorm(double m, const LamConst& L) {
    return (m >= L.m_low && m <= L.m_high) ? exp(-L.alpha * log(m)) : 0.0;
}
__device__ __forceinline__ double gauss_dev(double m, const LamConst& L) {
    double d = (m - L.mu) / L.sigma;
    return exp(-0.5 * d * d) / (L.sigma * 2.50662827463100050242);
}

// Inclusive block scan over `n` values in `a` (shared), in place; P = ceil(n / NT) consecutive values per thread.
__device__ void block_inclusive_scan(double* a, int n, double* scan_scratch) {
    int tid = threadIdx.x;
    int P = (n + kTabThreads - 1) / kTabThreads;
    int lo = tid * P, hi = min(lo + P, n);
    double run = 0.0;
    for (int i = lo; i < hi; ++i) {
        run += a[i];
        a[i] = run;
    }
    scan_scratch[tid] = run;
    __syncthreads();
    // serial exclusive scan of the 256 thread totals by one warp-friendly loop (fp64, tiny)
    if (tid == 0) {
        double acc = 0.0;
        for (int t = 0; t < kTabThreads; ++t) {
            double v = scan_scratch[t];
            scan_scratch[t] = acc;
            acc += v;
        }
    }
    __syncthreads();
    double off = scan_scratch[tid];
    for (int i = lo; i < hi; ++i) a[i] += off;
    __syncthreads();
}

// d_C at arbitrary z from the shared table (cubic Hermite, node slopes (c/H0)/E exact)
__device__ __forceinline__ double dc_hermite(const double* s_dc, double dz, int nz_nodes, double z, const LamConst& L) {
    double x = z / dz;
    int i = (int)x;
    i = max(0, min(i, nz_nodes - 2));
    double t = x - (double)i;
    double f0 = L.c_H0 * invE(i * dz, L.Om) * dz, f1 = L.c_H0 * invE((i + 1) * dz, L.Om) * dz;
    double t2 = t * t, omt = 1.0 - t;
    return (1.0 + 2.0 * t) * omt * omt * s_dc[i] + t2 * (3.0 - 2.0 * t) * s_dc[i + 1] + t * omt * omt * f0 - t2 * omt * f1;
}

// Build one ln d_L table (nodes in s_nodes[4][K+3], rows to global).
__device__ void build_dl_table(const DlGrid g, bool is_inj, int placement, const TabSmem& S, const double* s_dc,
                               const double* s_dl, double dz, int nz_nodes, double* s_nodes, Row* __restrict__ rows) {
    const LamConst& L = S.L;
    int NN = g.K + 3;
    for (int idx = threadIdx.x; idx < NN; idx += kTabThreads) {
        double target = exp(g.x0 + (idx - 1) * g.dx);
        // bisection over the monotone node values s_dl[0..nz_nodes-1]
        int lo = 0, hi = nz_nodes - 1;
        double z;
        if (target >= s_dl[hi]) {
            // beyond the (padded) table: linear continuation with the end slope; only ever touched by the
            // stencil of samples within 2 nodes of the table limit
            double zend = hi * dz, dce = s_dc[hi];
            double slope = dXi_of(zend, L) * (1.0 + zend) * dce + Xi_of(zend, L) * (dce + (1.0 + zend) * L.c_H0 * invE(zend, L.Om));
            z = zend + (target - s_dl[hi]) / slope;
        } else {
            while (hi - lo > 1) {
                int mid = (lo + hi) >> 1;
                if (s_dl[mid] <= target) lo = mid; else hi = mid;
            }
            double zl = lo * dz, zh = zl + dz;
            z = zl + dz * (target - s_dl[lo]) / (s_dl[lo + 1] - s_dl[lo]);
            for (int it = 0; it < 8; ++it) {
                double dc = dc_hermite(s_dc, dz, nz_nodes, z, L);
                double xi = Xi_of(z, L);
                double gval = xi * (1.0 + z) * dc - target;
                double gder = dXi_of(z, L) * (1.0 + z) * dc + xi * (dc + (1.0 + z) * L.c_H0 * invE(z, L.Om));
                double step = gval / gder;
                z -= step;
                z = fmin(fmax(z, zl), zh);
                if (fabs(step) < 1e-15 * (1.0 + z)) break;
            }
        }
        double u = log1p(z), a1 = 1.0 + z;
        double R = 1.0;
        if (is_inj || placement == CHIM_ON_SAMPLES) {
            double dc = (z <= (nz_nodes - 1) * dz) ? dc_hermite(s_dc, dz, nz_nodes, z, L)
                                                  : s_dc[nz_nodes - 1] + (z - (nz_nodes - 1) * dz) * L.c_H0 * invE(z, L.Om);
            double fE = L.c_H0 * invE(z, L.Om);
            double ddl = dXi_of(z, L) * a1 * dc + Xi_of(z, L) * (dc + a1 * fE);
            double J = a1 * a1 * a1 * fabs(ddl);                      // eq. (11)
            R = psi_of_u(u, L) / J;
            if (is_inj) R *= dc * dc * fE * L.vol_norm;               // u(z) of R6
        }
        s_nodes[0 * NN + idx] = z;
        s_nodes[1 * NN + idx] = u;
        s_nodes[2 * NN + idx] = 1.0 / a1;
        s_nodes[3 * NN + idx] = log(R);     // R > 0: psi, J and the volume factor are positive for z > 0
    }
    __syncthreads();
    // cubic through nodes k-1..k+2 expanded in t = tk - k; z and 1/(1+z) keep it (leading term split hi + lo),
    // ln(1+z) and log2 R drop t^3 by Chebyshev economisation on [0,1]: t^3 ~ 1.5 t^2 - 0.5625 t + 1/32 (error c3/32)
    for (int k = threadIdx.x; k < g.K + 2; k += kTabThreads) {
        double cf[4][4];
        int i0 = max(k - 1, 0), i3 = min(k + 2, NN - 1), i2 = min(k + 1, NN - 1);
#pragma unroll
        for (int c = 0; c < 4; ++c) {
            double f0 = s_nodes[c * NN + i0], f1 = s_nodes[c * NN + k], f2 = s_nodes[c * NN + i2], f3 = s_nodes[c * NN + i3];
            cf[c][0] = f1;
            cf[c][1] = -f0 / 3.0 - 0.5 * f1 + f2 - f3 / 6.0;
            cf[c][2] = 0.5 * f0 - f1 + 0.5 * f2;
            cf[c][3] = (f3 - f0) / 6.0 + 0.5 * (f1 - f2);
        }
        Row r;
        r.z_hi = (float)cf[0][0]; r.z_lo = (float)(cf[0][0] - (double)r.z_hi);
        r.z1 = (float)cf[0][1]; r.z2 = (float)cf[0][2]; r.z3 = (float)cf[0][3];
        r.a_hi = (float)cf[2][0]; r.a_lo = (float)(cf[2][0] - (double)r.a_hi);
        r.a1 = (float)cf[2][1]; r.a2 = (float)cf[2][2]; r.a3 = (float)cf[2][3];
        r.u0 = (float)(cf[1][0] + cf[1][3] / 32.0); r.u1 = (float)(cf[1][1] - 0.5625 * cf[1][3]); r.u2 = (float)(cf[1][2] + 1.5 * cf[1][3]);
        const double l2e = 1.4426950408889634074;
        r.r0 = (float)(l2e * (cf[3][0] + cf[3][3] / 32.0)); r.r1 = (float)(l2e * (cf[3][1] - 0.5625 * cf[3][3]));
        r.r2 = (float)(l2e * (cf[3][2] + 1.5 * cf[3][3]));
        rows[k] = r;
    }
    __syncthreads();
}

// W(m_low + mp) = int_{m_low}^{m_low+mp} m^beta S(m) dm from the cumulative panel table s_w + GL-8 on the partial panel.
__device__ double window_integral(const LamConst& L, const double* s_w, int n_win, double mp) {
    double x = mp * L.win_scale;
    int p = max(0, min((int)x, n_win - 1));
    double a0 = L.m_low + L.delta * p / n_win, b0 = L.m_low + mp;
    const int nsub = (p < 32) ? 8 : 1;
    double wdt = (b0 - a0) / nsub, acc = 0.0;
    for (int sub = 0; sub < nsub; ++sub) {
        double mid = a0 + (sub + 0.5) * wdt;
#pragma unroll
        for (int q = 0; q < kGLPanel; ++q) {
            double m = mid + 0.5 * wdt * c_glp_x[q];
            acc += c_glp_w[q] * exp(L.beta * log(m)) * smooth_S_dev(m, L);
        }
    }
    return s_w[p] + acc * 0.5 * wdt;
}

// Mass table (MassRow): nodes idx = 0..K+2 at y = lm0 + (idx-1)/inv_dlm, rows k = 0..K+1; node 1 is m1 = m_low
// exactly, node 0 lies below the support and is never used (the first interval takes a one-sided stencil).
__device__ void build_mass_table(const TableParams& P, const TabSmem& S, const double* s_w, double* s_nodes,
                                 MassRow* __restrict__ rows) {
    const LamConst& L = S.L;
    const int K = P.n_mass, NN = K + 3;
    const double dlm = 1.0 / L.inv_dlm;
    for (int idx = threadIdx.x; idx < NN; idx += kTabThreads) {
        // node idx sits where the sample kernels' fp32 coordinate ln m1 * tm_scale + mlow_tm equals idx: mlow_tm is rounded to a
        // float, so the nodes are shifted by that rounding (tm_shift rows, < 1e-7 in ln m) instead of the samples' coordinate
        // being wrong by it -- a bias common to every sample of a lambda otherwise.  (Node 1 then lies within 1e-7 m_low of m_low,
        // on either side: the asymptotic form below takes m' = m - m_low of either sign.)
        const double lm = L.lm0 + (idx - 1 - L.tm_shift) * dlm;
        const double m = (idx <= 1) ? L.m_low * exp(-L.tm_shift * dlm) : exp(lm);
        const double mp = m - L.m_low;
        // ln of the un-smoothed primary density / Z1: power law (no cut) + Gaussian, and the Gaussian alone
        const double dm = m - L.mu;
        const double lpl = L.a_pl - L.alpha * lm, lg = L.a_g - dm * dm * L.inv2s2;     // -inf if the component is absent
        const double hi = fmax(lpl, lg);
        double lna = (hi > -INFINITY) ? hi + log(exp(lpl - hi) + exp(lg - hi)) : -INFINITY, lnb = lg;
        // ln[ m'^2 S / C ]: above the window S = 1 and C continues in closed form; inside, C/S = rho m'^2
        double lnd;
        if (mp >= L.delta) {
            double pw = L.beta_is_m1 ? (lm - L.ln_mc) : (exp(L.bp1 * lm) - L.pow_mc_bp1) * L.inv_bp1;
            lnd = 2.0 * log(mp) - log(L.W_c + pw);
        } else {
            double x = mp * L.inv_delta, rho;
            if (x < 2e-3) rho = exp(L.beta * log(m)) * L.inv_delta * (1.0 - 2.0 * x);   // S underflows: asymptotic form
            else rho = window_integral(L, s_w, P.n_win, mp) / (smooth_S_dev(m, L) * mp * mp);
            lnd = -log(rho);
        }
        lna += lnd;
        lnb += lnd;
        s_nodes[idx] = (lna > kLnFloor) ? lna : kLnFloor;
        s_nodes[NN + idx] = (lnb > kLnFloor) ? lnb : kLnFloor;
    }
    __syncthreads();
    const double l2e = 1.4426950408889634074;
    for (int k = threadIdx.x; k < K + 2; k += kTabThreads) {
#pragma unroll
        for (int c = 0; c < 2; ++c) {
            const double* f = s_nodes + c * NN;
            double o[4];
            if (k <= 1) {   // forward stencil through nodes k..k+3 (k = 0 is never addressed; keep it finite)
                int b = max(k, 1);
                double g0 = f[b], g1 = f[b + 1], g2 = f[b + 2], g3 = f[b + 3];
                o[0] = g0;
                o[1] = -11.0 / 6.0 * g0 + 3.0 * g1 - 1.5 * g2 + g3 / 3.0;
                o[2] = g0 - 2.5 * g1 + 2.0 * g2 - 0.5 * g3;
                o[3] = (g3 - g0) / 6.0 + 0.5 * (g1 - g2);
            } else {
                int i3 = min(k + 2, NN - 1);
                double f0 = f[k - 1], f1 = f[k], f2 = f[k + 1], f3 = f[i3];
                o[0] = f1;
                o[1] = -f0 / 3.0 - 0.5 * f1 + f2 - f3 / 6.0;
                o[2] = 0.5 * f0 - f1 + 0.5 * f2;
                o[3] = (f3 - f0) / 6.0 + 0.5 * (f1 - f2);
            }
            rows[(size_t)c * (K + 2) + k] = make_float4((float)(l2e * o[0]), (float)(l2e * o[1]), (float)(l2e * o[2]), (float)(l2e * o[3]));
        }
    }
    __syncthreads();
}

__global__ void __launch_bounds__(kTabThreads) k_tables(const double* __restrict__ lam, int n_lambda, TableParams P,
                                                       LamConst* __restrict__ Lc, double* __restrict__ dc_tab,
                                                       Row* __restrict__ tab_ev, Row* __restrict__ tab_inj,
                                                       MassRow* __restrict__ mtab) {
    extern __shared__ __align__(16) unsigned char smem_raw[];
    TabSmem& S = *reinterpret_cast<TabSmem*>(smem_raw);
    const int nz_nodes = P.n_table + 1 + kZPad;
    double* s_dc = reinterpret_cast<double*>(smem_raw + ((sizeof(TabSmem) + 15) / 16) * 16);
    double* s_dl = s_dc + nz_nodes;
    double* s_w = s_dl + nz_nodes;                // [n_win + 1]
    double* s_nodes = s_w + (P.n_win + 1);        // [4][maxK + 3]
    const int l = blockIdx.x, tid = threadIdx.x;
    LamConst& L = S.L;
    const double dz = P.z_table_max / P.n_table;

    if (tid == 0) {
        const double* p = lam + (size_t)l * CHIM_N_LAMBDA_PARAMS;
        L.H0 = p[0]; L.Om = p[1]; L.Xi0 = p[2]; L.n = p[3]; L.alpha = p[4]; L.beta = p[5]; L.delta = p[6];
        L.m_low = p[7]; L.m_high = p[8]; L.mu = p[9]; L.sigma = p[10]; L.lg = p[11]; L.gamma = p[12];
        L.kappa = p[13]; L.zp = p[14];
        bool ok = (L.H0 > 0.0) && (L.Om > 0.0 && L.Om <= 1.0) && (L.Xi0 > 0.0) && (L.delta > 0.0) && (L.sigma > 0.0) &&
                  (L.lg >= 0.0 && L.lg <= 1.0) && (L.m_low > 0.0) && (L.m_high > L.m_low) && (L.zp > -1.0);
        for (int k = 0; k < CHIM_N_LAMBDA_PARAMS; ++k) ok = ok && isfinite(p[k]);
        L.flags = ok ? 0u : CHIM_FLAG_LAMBDA_DOMAIN;
        L.c_H0 = kCkms / L.H0;
        L.m_c = L.m_low + L.delta;
        L.inv2s2 = 0.5 / (L.sigma * L.sigma);
        L.bp1 = L.beta + 1.0;
        L.beta_is_m1 = fabs(L.bp1) < 1e-12;
        L.inv_bp1 = L.beta_is_m1 ? 0.0 : 1.0 / L.bp1;
        L.ln_mc = log(L.m_c);
        L.pow_mc_bp1 = exp(L.bp1 * L.ln_mc);
        L.gk = L.gamma + L.kappa;
        L.ln1pzp = log1p(L.zp);
        L.win_scale = P.n_win / L.delta;
        L.inv_delta = 1.0 / L.delta;
        L.lm0 = log(L.m_low);
        {   // the mass table spans [ln m_low, max(ln m_top, ln m_low + 1)]
            double top = fmax(P.ln_m_top, L.lm0 + 1.0);
            L.inv_dlm = (double)(float)((double)P.n_mass / ((top - L.lm0) * (1.0 + 1e-6)));   // exact in fp32 (LamF::tm_scale)
        }
        S.ibad = 0;
    }
    __syncthreads();
    if (L.flags) {
        if (tid == 0) Lc[l] = L;
        return;
    }

    // ---- d_C table: panel integrals (trapezoid + Euler-Maclaurin end term), prefix sum ----------------
    for (int i = tid; i < nz_nodes; i += kTabThreads) {
        if (i == 0) { s_dc[0] = 0.0; continue; }
        double za = (i - 1) * dz, zb = i * dz;
        double fa = invE(za, L.Om), fb = invE(zb, L.Om);
        s_dc[i] = 0.5 * dz * (fa + fb) + dz * dz / 12.0 * (dinvE(za, L.Om) - dinvE(zb, L.Om));
    }
    __syncthreads();
    block_inclusive_scan(s_dc, nz_nodes, S.scan);
    for (int i = tid; i < nz_nodes; i += kTabThreads) s_dc[i] *= L.c_H0;
    __syncthreads();
    // ---- d_L^gw nodes + monotonicity (analytic derivative > 0 at nodes 0..n_table, R16) ---------------
    int bad = 0;
    for (int i = tid; i < nz_nodes; i += kTabThreads) {
        double z = i * dz, dc = s_dc[i], xi = Xi_of(z, L);
        s_dl[i] = xi * (1.0 + z) * dc;
        double ddl = dXi_of(z, L) * (1.0 + z) * dc + xi * (dc + (1.0 + z) * L.c_H0 * invE(z, L.Om));
        if (!(ddl > 0.0) && i <= P.n_table) bad = 1;   // the rule covers nodes 0..n_table only
    }
    bad = __syncthreads_or(bad);
    if (bad) {
        if (tid == 0) { L.flags |= CHIM_FLAG_DL_NONMONOTONE; Lc[l] = L; }
        return;
    }
    if (dc_tab)
        for (int i = tid; i < nz_nodes; i += kTabThreads) dc_tab[(size_t)l * nz_nodes + i] = s_dc[i];

    // ---- mass-function normalisation Z1 (M2): 8 panels x 32 GL nodes on the window + closed-form tails -
    {
        double npl = (fabs(L.alpha - 1.0) < 1e-12)
                         ? log(L.m_high / L.m_low)
                         : (exp((1.0 - L.alpha) * log(L.m_high)) - exp((1.0 - L.alpha) * log(L.m_low))) / (1.0 - L.alpha);
        bool split = L.m_high < L.m_c;   // power law ends inside the window: integrate the two pieces apart
        int panel = tid >> 5, node = tid & 31;
        double a, b;
        if (split) {
            double lo = (panel < 4) ? L.m_low : L.m_high, hi = (panel < 4) ? L.m_high : L.m_c;
            int pp = panel & 3;
            a = lo + (hi - lo) * pp / 4.0; b = lo + (hi - lo) * (pp + 1) / 4.0;
        } else {
            a = L.m_low + L.delta * panel / 8.0; b = L.m_low + L.delta * (panel + 1) / 8.0;
        }
        double hw = 0.5 * (b - a), m = 0.5 * (a + b) + hw * c_glw_x[node];
        double plv = powerlaw_unnorm(m, L);
        if (split && panel >= 4) plv = 0.0;  // open at m_high from above
        double v[1] = {hw * c_glw_w[node] * ((1.0 - L.lg) * plv / npl + L.lg * gauss_dev(m, L)) * smooth_S_dev(m, L)};
        block_sum<kTabThreads, 1>(v, S.red);
        if (tid == 0) {
            double z1 = v[0];
            if (!split) {
                double tail = (fabs(L.alpha - 1.0) < 1e-12)
                                  ? log(L.m_high / L.m_c)
                                  : (exp((1.0 - L.alpha) * log(L.m_high)) - exp((1.0 - L.alpha) * log(L.m_c))) / (1.0 - L.alpha);
                z1 += (1.0 - L.lg) * tail / npl;
            }
            z1 += L.lg * 0.5 * erfc((L.m_c - L.mu) / (L.sigma * 1.41421356237309504880));
            L.Z1 = z1;
            L.a_pl = log((1.0 - L.lg) / (npl * z1));
            L.a_g = log(L.lg / (L.sigma * 2.50662827463100050242 * z1));
        }
    }
    // ---- window table (M4): W(m) = int m'^beta S by GL-8 per panel (the lowest 32 panels, where S varies
    //      super-exponentially, are split 8x), prefix sum, then rho = W / (S m'^2) at the nodes --------------
    for (int p = tid; p <= P.n_win; p += kTabThreads) {
        if (p == 0) { s_w[0] = 0.0; continue; }
        const int nsub = (p <= 32) ? 8 : 1;
        double a0 = L.m_low + L.delta * (p - 1) / P.n_win, wdt = L.delta / P.n_win / nsub, acc = 0.0;
        for (int sub = 0; sub < nsub; ++sub) {
            double mid = a0 + (sub + 0.5) * wdt;
#pragma unroll
            for (int q = 0; q < kGLPanel; ++q) {
                double m = mid + 0.5 * wdt * c_glp_x[q];
                acc += c_glp_w[q] * exp(L.beta * log(m)) * smooth_S_dev(m, L);
            }
        }
        s_w[p] = acc * 0.5 * wdt;
    }
    __syncthreads();
    block_inclusive_scan(s_w, P.n_win + 1, S.scan);
    if (tid == 0) {
        L.W_c = s_w[P.n_win];
        double dcc = dc_hermite(s_dc, dz, nz_nodes, P.z_cat_max, L);
        L.vol_norm = 3.0 / (dcc * dcc * dcc);
        L.dl_tabmax = s_dl[P.n_table];
        double lt = log(L.dl_tabmax);
        L.tkmax_ev = P.ev.K > 0 ? (lt - P.ev.x0) / P.ev.dx + 1.0 : 0.0;
        L.tkmax_inj = P.inj.K > 0 ? (lt - P.inj.x0) / P.inj.dx + 1.0 : 0.0;
        // fp32 constants of the sample kernels
        const double l2e = 1.4426950408889634074;
        LamF& F = L.F;
        F.mlow_hi = (float)L.m_low; F.mlow_lo = (float)(L.m_low - (double)F.mlow_hi);
        F.lm0_hi = (float)L.lm0; F.lm0_lo = (float)(L.lm0 - (double)F.lm0_hi);
        F.delta = (float)L.delta;
        F.two_dl2e = (float)(2.0 * L.delta * l2e); F.d2l2e = (float)(L.delta * L.delta * l2e);
        F.win_lo = (float)(L.delta * 1e-12); F.win_hi = (float)(L.delta * (1.0 - 1e-6));   // keeps f finite: log2 S down to -1e12 (the weights are carried as logs, R21)
        F.beta2 = (float)(L.beta * l2e); F.beta2_lo = (float)(L.beta * l2e - (double)F.beta2);
        F.mhigh_p = (float)(L.m_high - L.m_low);
        F.tm_scale = (float)L.inv_dlm; F.tm_max = (float)P.n_mass + 0.999f;
        F.tkmax_ev = (float)fmin(L.tkmax_ev, 1e9) * (1.0f - 1e-6f); F.tkmax_inj = (float)fmin(L.tkmax_inj, 1e9) * (1.0f - 1e-6f);
        F.zcat_hi = (float)P.z_cat_max; F.zcat_lo = (float)(P.z_cat_max - (double)F.zcat_hi);
        if (P.placement == CHIM_ON_SAMPLES) { F.gk2 = (float)(L.gk * l2e); F.cpsi = (float)(L.gk * l2e * L.ln1pzp); }
        else { F.gk2 = 0.f; F.cpsi = 100.f; }
        F.mlow_tm = (float)(1.0 - L.lm0 * L.inv_dlm);
        L.tm_shift = (double)F.mlow_tm - (1.0 - L.lm0 * L.inv_dlm);   // |.| < 2e-5 rows; build_mass_table moves its nodes by it
        F.tm_one = (float)(1.0 + L.tm_shift);
        F.gk2_inj = (float)(L.gk * l2e); F.cpsi_inj = (float)(L.gk * l2e * L.ln1pzp);
        F.tkmax_ev_q = (L.tkmax_ev >= 4095.9) ? 0xFFFFFFFFu : (L.tkmax_ev <= 0.0 ? 0u : (uint32_t)(L.tkmax_ev * (double)(1u << kTkFracBits)));
    }
    __syncthreads();
    build_mass_table(P, S, s_w, s_nodes, mtab + (size_t)l * 2 * (P.n_mass + 2));
    if (P.ev.K > 0)
        build_dl_table(P.ev, false, P.placement, S, s_dc, s_dl, dz, nz_nodes, s_nodes, tab_ev + (size_t)l * P.ev.rows());
    if (P.inj.K > 0)
        build_dl_table(P.inj, true, P.placement, S, s_dc, s_dl, dz, nz_nodes, s_nodes, tab_inj + (size_t)l * P.inj.rows());
    if (tid == 0) Lc[l] = L;
}

size_t tables_smem_bytes(const TableParams& P) {
    int nz_nodes = P.n_table + 1 + kZPad;
    int maxK = P.ev.K > P.inj.K ? P.ev.K : P.inj.K;
    size_t b = ((sizeof(TabSmem) + 15) / 16) * 16;
    size_t nodes = 4 * (size_t)(maxK + 3), mnodes = 2 * (size_t)(P.n_mass + 3);
    b += sizeof(double) * (2 * (size_t)nz_nodes + (P.n_win + 1) + (nodes > mnodes ? nodes : mnodes));
    return b;
}

cudaError_t launch_tables(const double* lam, int n_lambda, const TableParams& P, LamConst* Lc, double* dc_tab,
                          Row* tab_ev, Row* tab_inj, MassRow* mtab, cudaStream_t st) {
    size_t smem = tables_smem_bytes(P);
    cudaError_t e = cudaFuncSetAttribute(k_tables, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    if (e != cudaSuccess) return e;
    k_tables<<<n_lambda, kTabThreads, smem, st>>>(lam, n_lambda, P, Lc, dc_tab, tab_ev, tab_inj, mtab);
    return cudaGetLastError();
}

// Diagnostics: evaluate the event table at arbitrary d_L (single lambda).
// Local-polynomial fits for k_events (per (event, lambda)) and k_inject (per (chunk, lambda)): eight lanes per item.
// out[(l * n_ranges + r) * 4 * kPolyN ..]; items whose range is too wide (tk_h = 0), beyond the table or whose lambda is
// invalid are left untouched (the consumers test the same conditions and take the table path).
__global__ void __launch_bounds__(256) k_polyfit(const LamConst* __restrict__ Lc, const Row* __restrict__ tab, int tab_rows,
                                                 int n_lambda, int n_ranges, const double* __restrict__ tk_c,
                                                 const double* __restrict__ tk_h, const double* __restrict__ z_ref,
                                                 double z_ref_const, int is_inj, const double* __restrict__ pm,
                                                 const double* __restrict__ lnm1_lo, const double* __restrict__ lnm1_hi,
                                                 int n_mass, int mcap, double dx_tab, float* __restrict__ out) {
    // four items per warp, one per segment of eight lanes (the fp64 node evaluations occupy seven lanes of a segment)
    const long long item = ((long long)blockIdx.x * 8 + (threadIdx.x >> 5)) * 4 + ((threadIdx.x & 31) >> 3);
    const int sl = threadIdx.x & 7;
    bool valid = item < (long long)n_lambda * n_ranges;
    const int l = valid ? (int)(item % n_lambda) : 0, r = valid ? (int)(item / n_lambda) : 0;
    const LamConst& L = Lc[l];
    const double h = tk_h[r], c = tk_c[r];
    valid = valid && !L.flags && (h > 0.0) && (c + h < (is_inj ? L.tkmax_inj : L.tkmax_ev));
    float* o = out + ((size_t)l * n_ranges + r) * (4 * kPolyN);
    // the Madau-Dickinson turnover log2(1 + ((1+z)/(1+z_p))^(gamma+kappa)) is kept out of the fitted polynomial r (its poles sit
    // ~0.5 from the real axis in ln(1+z)) -- except for injection chunks narrower than 0.2 in ln d_L, where degree 6 takes it
    // to < 1e-9 and k_inject saves two MUFU per injection (slot 26 of the record: 1 = folded)
    const bool fold = is_inj && h * dx_tab <= 0.1;
    double r0_lo = 0.0;
    fit_polys(L, tab + (size_t)l * tab_rows, tab_rows - 2, c, h, z_ref ? z_ref[r] : z_ref_const, !fold && (is_inj || L.F.gk2 != 0.f), pm, o, valid,
              &r0_lo);
    if (is_inj) {
        __syncwarp();
        // slot 27 (free for chunks): what the fp32 constant term of r lost -- k_inject scales the chunk's sums by 2^r0_lo
        if (valid && sl == 0) { o[26] = __int_as_float(fold ? 1 : 0); o[27] = (float)r0_lo; }
    }
    if (lnm1_lo) {
        // k_events: the rows of the mass table the event can address, ln m1 = ln m1d - u, u = ln(1+z) between the ends of the
        // event's range (the fitted polynomial at t = -1, +1), so that the CTA can issue its TMA copy at once.  Slots 26, 27 of
        // the record (the unused degree-6 terms of u and a): first staged row, and the row count (negative: does not fit)
        __syncwarp();
        const float cu = (valid && sl < kPolyN - 1) ? o[2 * kPolyN + 2 * sl] : 0.f;          // u_n
        float up = cu, um = (sl & 1) ? -cu : cu;
#pragma unroll
        for (int k = 4; k > 0; k >>= 1) { up += __shfl_xor_sync(0xffffffffu, up, k); um += __shfl_xor_sync(0xffffffffu, um, k); }
        if (valid && sl == 0) {
            const double u_lo = fmin((double)um, (double)up) - 1e-4, u_hi = fmax((double)um, (double)up) + 1e-4;
            const int ma = max(1, min((int)fma(lnm1_lo[r] - u_hi - L.lm0, L.inv_dlm, 1.0), n_mass));
            const int mb = max(1, min((int)fma(lnm1_hi[r] - u_lo - L.lm0, L.inv_dlm, 1.0), n_mass));
            int mlo = ma - 1 + max(0, (mb - ma + 3 - mcap) / 2);                          // wider than the stage: keep the centre
            mlo = max(0, min(mlo, n_mass + 2 - mcap));
            const int nrow = min(mcap, mb + 3 - mlo);
            o[26] = __int_as_float(mlo);
            o[27] = __int_as_float((mb - ma + 3 <= mcap) ? nrow : -nrow);
        }
    }
}

cudaError_t launch_polyfit(const LamConst* Lc, const Row* tab, int tab_rows, int n_lambda, int n_ranges, const double* tk_c,
                           const double* tk_h, const double* z_ref, double z_ref_const, bool is_inj, const double* pm,
                           const double* lnm1_lo, const double* lnm1_hi, int n_mass, int mcap, double dx_tab, float* out, cudaStream_t st) {
    const long long items = (long long)n_lambda * n_ranges;
    if (items <= 0) return cudaSuccess;
    k_polyfit<<<(unsigned)((items + 31) / 32), 256, 0, st>>>(Lc, tab, tab_rows, n_lambda, n_ranges, tk_c, tk_h, z_ref, z_ref_const,
                                                            is_inj ? 1 : 0, pm, lnm1_lo, lnm1_hi, n_mass, mcap, dx_tab, out);
    return cudaGetLastError();
}

// ---- p_cat from galaxy lists (eq. 8; one-off, before the hot path; R22) -----------------------
// One CTA per line of sight (event or pixel).  dV_c/dz is needed up to a constant only (it cancels against the per-galaxy
// normalisation): V(z) = I(z)^2 / E(z), I(z) = int_0^z dz'/E by one 32-node Gauss-Legendre panel.  fp64 throughout.
__device__ __forceinline__ double pcat_vol(double z, double Om) {
    double I = 0.0;
    const double hz = 0.5 * z;
#pragma unroll 4
    for (int q = 0; q < kGLWin; ++q) {
        const double a = 1.0 + hz * (1.0 + c_glw_x[q]);
        I += c_glw_w[q] * rsqrt(Om * a * a * a + 1.0 - Om);
    }
    I *= hz;
    const double a = 1.0 + z;
    return I * I * rsqrt(Om * a * a * a + 1.0 - Om);
}

__global__ void __launch_bounds__(256) k_pcat(double Om, const int64_t* __restrict__ gal_off, const double* __restrict__ zt,
                                              const double* __restrict__ st, const double* __restrict__ wg,
                                              const int64_t* __restrict__ grid_off, const double* __restrict__ zg,
                                              double* __restrict__ coef, double* __restrict__ out) {
    __shared__ double red[256 / 32];
    __shared__ double s_sw;
    const int e = blockIdx.x, tid = threadIdx.x;
    const int64_t g0 = gal_off[e], g1 = gal_off[e + 1], p0 = grid_off[e], p1 = grid_off[e + 1];
    // per galaxy: Z_g = int N(z; zt, st) V(z) dz over [max(0, zt - 10 st), zt + 10 st], 8 panels of 32 nodes
    double sw = 0.0;
    for (int64_t g = g0 + tid; g < g1; g += 256) {
        const double m = zt[g], s = st[g], w = wg ? wg[g] : 1.0;
        const double lo = fmax(0.0, m - 10.0 * s), hi = m + 10.0 * s, hw = 0.5 * (hi - lo) / 8.0;
        double Z = 0.0;
        for (int p = 0; p < 8; ++p) {
            const double mid = lo + (2 * p + 1) * hw;
            double acc = 0.0;
            for (int q = 0; q < kGLWin; ++q) {
                const double z = mid + hw * c_glw_x[q], u = (z - m) / s;
                acc += c_glw_w[q] * exp(-0.5 * u * u) * pcat_vol(z, Om);
            }
            Z += acc * hw;
        }
        coef[g] = w / Z;          // (the Gaussian's 1/(s sqrt(2 pi)) is common to N and Z_g: it cancels)
        sw += w;
    }
    sw = warp_sum(sw);
    if ((tid & 31) == 0) red[tid >> 5] = sw;
    __syncthreads();              // also publishes coef[] (same CTA)
    if (tid == 0) {
        double a = 0.0;
        for (int k = 0; k < 256 / 32; ++k) a += red[k];
        s_sw = a;
    }
    __syncthreads();
    const double inv_sw = 1.0 / s_sw;
    for (int64_t i = p0 + tid; i < p1; i += 256) {
        const double z = zg[i];
        double acc = 0.0;
        for (int64_t g = g0; g < g1; ++g) {
            const double u = (z - zt[g]) / st[g];
            if (fabs(u) < 39.0) acc += coef[g] * exp(-0.5 * u * u);      // exp(-760) underflows fp64
        }
        out[i] = acc * inv_sw * pcat_vol(z, Om);
    }
}

cudaError_t launch_pcat(double Om, int n_los, const int64_t* gal_off, const double* zt, const double* st, const double* wg,
                        const int64_t* grid_off, const double* zg, double* coef, double* out, cudaStream_t st_) {
    if (n_los <= 0) return cudaSuccess;
    k_pcat<<<n_los, 256, 0, st_>>>(Om, gal_off, zt, st, wg, grid_off, zg, coef, out);
    return cudaGetLastError();
}

// ---- completeness terms of p_gal (PAPER.md:58 eq. 7, :65 eq. 9, :67 eq. 10; one-off, R25) --------------------
// One CTA per line of sight, after k_pcat has written p_cat into `out`:
//   f_R = int_0^zmax P_compl(z) u(z) dz,  u = (dV_c/dz)/V_c(zmax) = 3 I(z)^2 / (E(z) I(zmax)^3),  I(z) = int_0^z dz'/E
//   p_gal(z) = f_R p_cat(z) + [1 - P_compl(z)] u(z)  (u = 0 beyond zmax)
// P_compl: nc nodes per line of sight, linear in between, constant beyond the ends.  f_R: one 32-node Gauss-Legendre panel on
// every stretch between consecutive nodes (the integrand is a linear function times a smooth one there).  fp64 throughout.
__device__ __forceinline__ double pcat_I(double z, double Om) {
    double I = 0.0;
    const double hz = 0.5 * z;
#pragma unroll 4
    for (int q = 0; q < kGLWin; ++q) {
        const double a = 1.0 + hz * (1.0 + c_glw_x[q]);
        I += c_glw_w[q] * rsqrt(Om * a * a * a + 1.0 - Om);
    }
    return I * hz;
}
__device__ __forceinline__ double compl_at(const double* __restrict__ zc, const double* __restrict__ pc, int nc, double z) {
    if (z <= zc[0]) return pc[0];
    if (z >= zc[nc - 1]) return pc[nc - 1];
    int lo = 0, hi = nc - 1;                       // zc[lo] <= z < zc[hi]
    while (hi - lo > 1) { const int mid = (lo + hi) >> 1; if (zc[mid] <= z) lo = mid; else hi = mid; }
    const double t = (z - zc[lo]) / (zc[lo + 1] - zc[lo]);
    return pc[lo] + t * (pc[lo + 1] - pc[lo]);
}
__global__ void __launch_bounds__(256) k_pgal(double Om, double zmax, const int64_t* __restrict__ compl_off,
                                              const double* __restrict__ zc_all, const double* __restrict__ pc_all,
                                              const int64_t* __restrict__ grid_off, const double* __restrict__ zg,
                                              double* __restrict__ out, double* __restrict__ fr_out) {
    __shared__ double red[256 / 32];
    __shared__ double s_fr;
    const int e = blockIdx.x, tid = threadIdx.x;
    const int64_t c0 = compl_off[e], p0 = grid_off[e], p1 = grid_off[e + 1];
    const int nc = (int)(compl_off[e + 1] - c0);
    const double* zc = zc_all + c0;
    const double* pc = pc_all + c0;
    const double Im = pcat_I(zmax, Om), inv_v = 3.0 / (Im * Im * Im);
    double acc = 0.0;
    for (int idx = tid; idx < (nc + 1) * kGLWin; idx += 256) {
        const int k = idx / kGLWin, q = idx - k * kGLWin;
        const double a = fmin((k == 0) ? 0.0 : zc[k - 1], zmax), b = fmin((k < nc) ? zc[k] : zmax, zmax);
        if (b > a) {
            const double hw = 0.5 * (b - a), z = a + hw * (1.0 + c_glw_x[q]);
            acc += c_glw_w[q] * hw * compl_at(zc, pc, nc, z) * pcat_vol(z, Om) * inv_v;
        }
    }
    acc = warp_sum(acc);
    if ((tid & 31) == 0) red[tid >> 5] = acc;
    __syncthreads();
    if (tid == 0) {
        double a = 0.0;
        for (int k = 0; k < 256 / 32; ++k) a += red[k];
        s_fr = a;
        if (fr_out) fr_out[e] = a;
    }
    __syncthreads();
    const double fr = s_fr;
    for (int64_t i = p0 + tid; i < p1; i += 256) {
        const double z = zg[i], u = (z <= zmax) ? pcat_vol(z, Om) * inv_v : 0.0;
        out[i] = fr * out[i] + (1.0 - compl_at(zc, pc, nc, z)) * u;
    }
}

cudaError_t launch_pgal(double Om, double zmax, int n_los, const int64_t* compl_off, const double* zc, const double* pc,
                        const int64_t* grid_off, const double* zg, double* out, double* fr_out, cudaStream_t st_) {
    if (n_los <= 0) return cudaSuccess;
    k_pgal<<<n_los, 256, 0, st_>>>(Om, zmax, compl_off, zc, pc, grid_off, zg, out, fr_out);
    return cudaGetLastError();
}

__global__ void k_table_lookup(const LamConst* __restrict__ Lc, const Row* __restrict__ tab, DlGrid g, int64_t n,
                               const double* __restrict__ dL, double z_table_max, double* __restrict__ z_out,
                               double* __restrict__ r_out) {
    int64_t i = blockIdx.x * (int64_t)blockDim.x + threadIdx.x;
    if (i >= n) return;
    const LamConst& L = Lc[0];
    double z = NAN, r = NAN;
    if (L.flags == 0) {
        double tk = (log(dL[i]) - g.x0) / g.dx + 1.0;
        if (tk > L.tkmax_ev) { z = z_table_max; r = 0.0; }
        else if (tk >= 1.0 && tk < g.K + 1.0) {
            int k = (int)tk;
            double t = tk - k;
            const Row& q = tab[k];
            const double tt = (double)(float)t;
            z = (double)q.z_hi + ((double)q.z_lo + tt * ((double)q.z1 + tt * ((double)q.z2 + tt * (double)q.z3)));
            r = exp2((double)q.r0 + tt * ((double)q.r1 + tt * (double)q.r2));
        }
    }
    if (z_out) z_out[i] = z;
    if (r_out) r_out[i] = r;
}

cudaError_t launch_table_lookup(const LamConst* Lc, const Row* tab, DlGrid g, int64_t n, const double* dL,
                                double z_table_max, double* z_out, double* r_out, cudaStream_t st) {
    if (n <= 0) return cudaSuccess;
    k_table_lookup<<<(unsigned)((n + 255) / 256), 256, 0, st>>>(Lc, tab, g, n, dL, z_table_max, z_out, r_out);
    return cudaGetLastError();
}

}  // namespace chim
