// k_events.cu -- steps S2 + S3 + S4 fused: one CTA per (event, lambda).
//
//   S2  per posterior sample: z_j from the per-lambda table, source masses, population weight w_j
//       (sample_weight, chim_internal.cuh), weighted moments -> Scott bandwidth h (R3), all in fp64.
//       z_j and w_j never leave shared memory.
//   S3  Gaussian KDE on the event's redshift grid (eq. 19, R2): grid points in registers (one per
//       lane, 32-point tiles per warp), samples broadcast from shared memory, fp32 FADD/FMUL + MUFU.EX2 +
//       FFMA per pair, short fp32 partial sums flushed into fp64.  Samples are sorted in z (they are sorted
//       in d_L at init and d_L^gw is monotone), so each tile only visits the samples within t*h of it (R9).
//   S4  I_i = sum_g K(z_g) q_g, q_g = p_gal(z_g) x trapezoid weight (eq. 14): warp shuffles +
//       block reduction in fp64, log I_i written per (lambda, event).
#include "chim_internal.cuh"

namespace chim {

constexpr int kEvThreads = 256;
constexpr int kFlush = 256;   // samples per fp32 partial sum before it is added to the fp64 accumulator

__device__ __forceinline__ float ex2_approx(float x) {
    float y;
    asm("ex2.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x));
    return y;
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
    int tile_counter;
};

__global__ void __launch_bounds__(kEvThreads) k_events(EventKernelParams P) {
    extern __shared__ __align__(16) unsigned char smem_raw[];
    EvSmem& S = *reinterpret_cast<EvSmem*>(smem_raw);
    double* zbuf = reinterpret_cast<double*>(smem_raw + ((sizeof(EvSmem) + 15) / 16) * 16);
    const int tid = threadIdx.x, lane = tid & 31, wid = tid >> 5;

    int l, ev;
    if (P.dbg_event >= 0) { l = blockIdx.x; ev = P.dbg_event; }
    else { l = blockIdx.x % P.n_lambda; ev = blockIdx.x / P.n_lambda; }   // lambda fastest: CTAs in flight share an event
    const int64_t s0 = P.ev.sample_off[ev], g0 = P.ev.grid_off[ev];
    const int ns = (int)(P.ev.sample_off[ev + 1] - s0), nz = (int)(P.ev.grid_off[ev + 1] - g0);
    double* wbuf = zbuf + P.ev.max_ns;
    float2* pk = reinterpret_cast<float2*>(zbuf);   // aliases zbuf slot j (same thread reads then writes slot j)
    double* out = (P.dbg_event >= 0) ? P.logI + l : P.logI + (size_t)l * P.ev.n_events + ev;

    {   // stage the per-lambda constants in shared memory
        const int nw = sizeof(LamConst) / 4;
        const uint32_t* src = reinterpret_cast<const uint32_t*>(P.Lc + l);
        uint32_t* dst = reinterpret_cast<uint32_t*>(&S.L);
        for (int i = tid; i < nw; i += kEvThreads) dst[i] = src[i];
        if (tid == 0) S.tile_counter = 0;
    }
    __syncthreads();
    const LamConst& L = S.L;
    if (L.flags) {   // invalid lambda: NaN
        if (tid == 0) *out = NAN;
        return;
    }
    const Row* tab = P.tab + (size_t)l * P.tab_rows;
    const double* wtab = P.wtab + (size_t)l * (P.n_win + 1);
    const double z0 = P.ev.z0[ev];

    // ---- S2: weights + centred moments -----------------------------------------------------------------
    double mom[4] = {0.0, 0.0, 0.0, 0.0};   // sum w, sum w^2, sum w z', sum w z'^2
    int oor = 0;
    for (int j = tid; j < ns; j += kEvThreads) {
        double2 A = P.ev.recA[s0 + j], B = P.ev.recB[s0 + j], C = P.ev.recC[s0 + j];
        double z, w;
        bool o;
        sample_weight(L, tab, P.tab_rows, wtab, P.n_win, L.tkmax_ev, P.z_table_max, A.x, A.y, B.x, B.y, C.x, C.y, z, w, o);
        oor |= (int)o;
        double zc = z - z0;
        zbuf[j] = zc;
        wbuf[j] = w;
        mom[0] += w;
        mom[1] += w * w;
        mom[2] += w * zc;
        mom[3] += w * zc * zc;
        if (P.dbg_z) {
            int jo = P.ev.perm[s0 + j];
            P.dbg_z[jo] = z;
            P.dbg_w[jo] = w * exp(P.ln_shift[ev]);
        }
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
        if (P.dbg_K) for (int g = tid; g < nz; g += kEvThreads) P.dbg_K[g] = 0.0;
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
    const double sc = sqrt(kHalfLog2e) / h;   // x = z' * sc  =>  exp(-d^2/2h^2) = 2^(-(dx)^2)
    const double wscale = (double)ns / sw;    // weights normalised to mean 1 before rounding to fp32
    for (int j = tid; j < ns; j += kEvThreads) {
        double zc = zbuf[j], w = wbuf[j];
        pk[j] = make_float2((float)(zc * sc), (float)(w * wscale));
    }
    __syncthreads();

    // ---- S3 + S4: tiles of 32 grid points per warp -----------------------------------------------------
    const float T = (P.cutoff > 0.0) ? (float)(P.cutoff * sqrt(kHalfLog2e)) : INFINITY;
    const float x_min = pk[0].x, x_max = pk[ns - 1].x;
    const int n_tiles = (nz + 31) / 32;
    const double* zc_g = P.ev.zc + g0;
    const double* q_g = P.ev.qg + g0;
    const double knorm = (sw / ns) / ((double)ns * h * 2.50662827463100050242);
    double wsum = 0.0;                 // this warp's sum_g K q (lane 0 holds the reduced value per tile)
    unsigned long long pairs = 0;
    for (;;) {
        int tile = 0;
        if (lane == 0) tile = atomicAdd(&S.tile_counter, 1);
        tile = __shfl_sync(0xffffffffu, tile, 0);
        if (tile >= n_tiles) break;
        const int g = tile * 32 + lane;
        const bool valid = g < nz;
        const int gc = valid ? g : nz - 1;
        const float xg = (float)(zc_g[gc] * sc);
        const float x_lo = __shfl_sync(0xffffffffu, xg, 0);
        const float x_hi = __shfl_sync(0xffffffffu, xg, min(31, nz - 1 - tile * 32));
        double accd = 0.0;
        if (!(x_hi + T < x_min || x_lo - T > x_max)) {
            // sample window [j_lo, j_hi): x_j in [x_lo - T, x_hi + T]  (warp-uniform binary searches)
            int j_lo = 0, j_hi = ns;
            if (T < INFINITY) {
                const float lo_key = x_lo - T, hi_key = x_hi + T;
                int a = 0, b = ns;
                while (a < b) { int m = (a + b) >> 1; if (pk[m].x < lo_key) a = m + 1; else b = m; }
                j_lo = a;
                b = ns;
                while (a < b) { int m = (a + b) >> 1; if (pk[m].x <= hi_key) a = m + 1; else b = m; }
                j_hi = a;
            }
            pairs += (unsigned long long)(j_hi - j_lo) * 32ull;
            for (int jb = j_lo; jb < j_hi; jb += kFlush) {
                const int je = min(jb + kFlush, j_hi);
                float acc0 = 0.f, acc1 = 0.f;
                int j = jb;
                for (; j + 4 <= je; j += 4) {
                    float2 s0_ = pk[j], s1_ = pk[j + 1], s2_ = pk[j + 2], s3_ = pk[j + 3];
                    float d0 = xg - s0_.x, d1 = xg - s1_.x, d2 = xg - s2_.x, d3 = xg - s3_.x;
                    acc0 = fmaf(s0_.y, ex2_approx(-d0 * d0), acc0);
                    acc1 = fmaf(s1_.y, ex2_approx(-d1 * d1), acc1);
                    acc0 = fmaf(s2_.y, ex2_approx(-d2 * d2), acc0);
                    acc1 = fmaf(s3_.y, ex2_approx(-d3 * d3), acc1);
                }
                for (; j < je; ++j) {
                    float2 s_ = pk[j];
                    float d = xg - s_.x;
                    acc0 = fmaf(s_.y, ex2_approx(-d * d), acc0);
                }
                accd += (double)(acc0 + acc1);
            }
        }
        double val = 0.0;
        if (valid) {
            double q = q_g[g];
            if (P.placement == CHIM_ON_GRID)
                q *= grid_factor(L, P.dc_tab + (size_t)l * (P.n_table + 1 + kZPad), P.n_table + 1 + kZPad,
                                 P.z_table_max / P.n_table, zc_g[g] + z0);
            val = accd * q;
            if (P.dbg_K) P.dbg_K[g] = accd * knorm * exp(P.ln_shift[ev]);
        }
        wsum += warp_sum(val);
    }
    double tot[1] = {lane == 0 ? wsum : 0.0};
    block_sum<kEvThreads, 1>(tot, S.red);
    if (lane == 0 && pairs) atomicAdd(P.stats, pairs);
    if (tid == 0) {
        double I = tot[0] * knorm;
        if (I > 0.0) *out = log(I) + P.ln_shift[ev];
        else if (I == 0.0) { *out = -INFINITY; atomicOr(P.flags + l, CHIM_FLAG_EVENT_ZERO); }
        else *out = NAN;
    }
}

size_t events_smem_bytes(int max_ns) {
    return ((sizeof(EvSmem) + 15) / 16) * 16 + 2 * sizeof(double) * (size_t)max_ns;
}

cudaError_t launch_events(const EventKernelParams& P, cudaStream_t st) {
    size_t smem = events_smem_bytes(P.ev.max_ns);
    cudaError_t e = cudaFuncSetAttribute(k_events, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    if (e != cudaSuccess) return e;
    long long nb = (P.dbg_event >= 0) ? P.n_lambda : (long long)P.n_lambda * P.ev.n_events;
    if (nb <= 0) return cudaSuccess;
    k_events<<<(unsigned)nb, kEvThreads, smem, st>>>(P);
    return cudaGetLastError();
}

}  // namespace chim
