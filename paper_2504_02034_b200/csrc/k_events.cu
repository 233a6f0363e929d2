// k_events.cu -- steps S2 + S3 + S4 fused: one CTA per (event, lambda).
//
//   S2  per posterior sample: z_j from the per-lambda table, source masses, population weight w_j
//       (sample_weight, chim_internal.cuh), weighted moments -> Scott bandwidth h (R3), all in fp64.
//       z_j and w_j never leave shared memory.
//   S3  Gaussian KDE on the event's redshift grid (eq. 19, R2): grid points in registers (one per
//       lane, 32-point tiles), samples broadcast from shared memory two per 128-bit load, fp32 FFMA +
//       MUFU.EX2 + FADD per pair (expanded square around the tile centre, log2 w_j folded into the per-sample
//       constant), fp32 partial sums over <= 256 samples flushed into fp64.  Samples are sorted
//       in z (they are sorted in d_L at init and d_L^gw is monotone), so each tile only visits the samples within
//       t*h of it (R9).  Work items are (tile, 256-sample chunk), handed to warps through a shared counter so
//       that the CTA's tail stays short.
//   S4  I_i = sum_g K(z_g) q_g, q_g = p_gal(z_g) x trapezoid weight (eq. 14): warp shuffles +
//       block reduction in fp64, log I_i written per (lambda, event).
#include "chim_internal.cuh"

namespace chim {

constexpr int kEvThreads = 256;
constexpr int kFlush = 256;   // samples per work item = length of one fp32 partial sum before it goes to fp64
constexpr float kMaxHalfWidth = 2.5f;   // widest tile (half width, scaled units) handled by the expanded-square loop

__device__ __forceinline__ float lg2_approx(float x) {
    float y;
    asm("lg2.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x));
    return y;
}
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

// the float region after wbuf holds zf[ns_pad] during S2 and the per-warp scratch (kFlush float2 per warp) afterwards
__host__ __device__ inline size_t ev_float_region(size_t ns_pad) {
    size_t scratch = (size_t)(kEvThreads / 32) * kFlush * 2;
    return ns_pad > scratch ? ns_pad : scratch;
}
struct EvSmem {
    LamConst L;
    double red[4 * (kEvThreads / 32)];
    int item_counter;
    int n_items;
};

// shared-memory layout after EvSmem: wbuf double[max_ns] (re-used in place as float2 pk[max_ns]) | zf float[max_ns] |
// tile_jlo int[max_tiles] | tile_jhi int[max_tiles] | tile_cum int[max_tiles + 1]
__global__ void __launch_bounds__(kEvThreads, 3) k_events(EventKernelParams P) {
    extern __shared__ __align__(16) unsigned char smem_raw[];
    EvSmem& S = *reinterpret_cast<EvSmem*>(smem_raw);
    double* wbuf = reinterpret_cast<double*>(smem_raw + ((sizeof(EvSmem) + 15) / 16) * 16);
    const int ns_pad = (P.ev.max_ns + 3) & ~3;
    float* zf = reinterpret_cast<float*>(wbuf + ns_pad);
    const int max_tiles = (P.ev.max_nz + 31) / 32;
    int* tile_jlo = reinterpret_cast<int*>(zf + ev_float_region(ns_pad));
    int* tile_jhi = tile_jlo + max_tiles;
    int* tile_cum = tile_jhi + max_tiles;
    float2* pk = reinterpret_cast<float2*>(wbuf);   // aliases wbuf slot j (same thread reads then writes slot j)
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
        if (tid == 0) S.item_counter = 0;
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
#pragma unroll 1
    for (int j = tid; j < ns; j += kEvThreads) {
        double2 A = P.ev.recA[s0 + j], B = P.ev.recB[s0 + j], C = P.ev.recC[s0 + j];
        double z, w;
        bool o;
        sample_weight(L, tab, P.tab_rows, wtab, P.n_win, L.tkmax_ev, P.z_table_max, A.x, A.y, B.x, B.y, C.x, C.y, z, w, o);
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
    const double sc = sqrt(kHalfLog2e) / h;   // x = z' * sc  =>  exp(-d^2/2h^2) = 2^(-(dx)^2)
    const double wscale = (double)ns / sw;    // weights normalised to mean 1 before rounding to fp32
    const float scf = (float)sc;
    for (int j = tid; j < ns; j += kEvThreads) {   // pk[j] = {x_j, log2 of the normalised weight}; log2(0) = -inf
        float x = zf[j] * scf;
        double w = wbuf[j];
        pk[j] = make_float2(x, lg2_approx((float)(w * wscale)));
    }
    __syncthreads();   // zf is dead from here on: its storage becomes the per-warp scratch of the pair loop

    // ---- tile windows, in parallel: tile t = grid points [32t, 32t+32), samples with x_j in [x_lo - T, x_hi + T] --
    const float T = (P.cutoff > 0.0) ? (float)(P.cutoff * sqrt(kHalfLog2e)) : INFINITY;
    const int n_tiles = (nz + 31) / 32;
    const double* zc_g = P.ev.zc + g0;
    const double* q_g = P.ev.qg + g0;
    unsigned long long pairs = 0;
    for (int t = tid; t < n_tiles; t += kEvThreads) {
        int j_lo = 0, j_hi = ns;
        if (T < INFINITY) {
            const float lo_key = (float)zc_g[t * 32] * scf - T, hi_key = (float)zc_g[min(t * 32 + 31, nz - 1)] * scf + T;
            int a = 0, b = ns;
            while (a < b) { int m = (a + b) >> 1; if (pk[m].x < lo_key) a = m + 1; else b = m; }
            j_lo = a;
            b = ns;
            while (a < b) { int m = (a + b) >> 1; if (pk[m].x <= hi_key) a = m + 1; else b = m; }
            j_hi = max(a, j_lo);
        }
        tile_jlo[t] = j_lo;
        tile_jhi[t] = j_hi;
        pairs += (unsigned long long)(j_hi - j_lo) * 32ull;
    }
    __syncthreads();
    if (tid < 32) {   // exclusive scan of the chunk counts (warp 0)
        int run = 0;
        for (int base = 0; base < n_tiles; base += 32) {
            int t = base + lane;
            int c = (t < n_tiles) ? (tile_jhi[t] - tile_jlo[t] + kFlush - 1) / kFlush : 0;
            int inc = c;
#pragma unroll
            for (int o = 1; o < 32; o <<= 1) { int v = __shfl_up_sync(0xffffffffu, inc, o); if (lane >= o) inc += v; }
            if (t < n_tiles) tile_cum[t] = run + inc - c;
            run += __shfl_sync(0xffffffffu, inc, 31);
        }
        if (lane == 0) { tile_cum[n_tiles] = run; S.n_items = run; }
    }
    __syncthreads();

    // ---- S3 + S4: work items = (tile, chunk of <= kFlush samples), one grid point per lane ----------------
    // With c the tile centre, x' = x - c:  -(xg - xj)^2 + log2 w_j = -xg'^2 + [ xg' (2 xj') + (log2 w_j - xj'^2) ].
    // The warp first writes {2 xj', log2 w_j - xj'^2} for its chunk into its scratch, so that the pair loop is
    // FFMA (argument) -> MUFU.EX2 -> FADD per pair; the lane factor 2^(-xg'^2) is applied once per item.  Tiles
    // wider than kMaxHalfWidth (in units of h sqrt(2 ln 2)) -- a bandwidth far below the grid spacing -- take the
    // direct path, where the products would lose fp32 precision.
    const int n_items = S.n_items;
    float2* scratch = reinterpret_cast<float2*>(zf) + (tid >> 5) * kFlush;
    const float4* scratch4 = reinterpret_cast<const float4*>(scratch);
    double lsum = 0.0;                 // this lane's sum over its (g, j) pairs of w_j e_gj q_g
    for (;;) {
        int item = 0;
        if (lane == 0) item = atomicAdd(&S.item_counter, 1);
        item = __shfl_sync(0xffffffffu, item, 0);
        if (item >= n_items) break;
        int a = 0, b = n_tiles;        // largest tile with tile_cum[tile] <= item
        while (b - a > 1) { int m = (a + b) >> 1; if (tile_cum[m] <= item) a = m; else b = m; }
        const int tile = a;
        const int jb = tile_jlo[tile] + (item - tile_cum[tile]) * kFlush;
        const int je = min(jb + kFlush, tile_jhi[tile]);
        const int g = tile * 32 + lane;
        const bool valid = g < nz;
        const float xg = (float)zc_g[valid ? g : nz - 1] * scf;
        const float x_lo = __shfl_sync(0xffffffffu, xg, 0), x_hi = __shfl_sync(0xffffffffu, xg, 31);
        const float c = 0.5f * (x_lo + x_hi);
        float acc;
        if (0.5f * (x_hi - x_lo) <= kMaxHalfWidth) {
            const int cnt = je - jb;
#pragma unroll
            for (int i = 0; i < kFlush / 32; ++i) {
                const int jj = lane + 32 * i;
                if (jj < ((cnt + 7) & ~7)) {
                    float2 sj = (jj < cnt) ? pk[jb + jj] : make_float2(c, -INFINITY);
                    const float xp = sj.x - c;
                    scratch[jj] = make_float2(xp + xp, fmaf(-xp, xp, sj.y));
                }
            }
            __syncwarp();
            const float xgp = xg - c;
            float acc0 = 0.f, acc1 = 0.f, acc2 = 0.f, acc3 = 0.f;
            const int n8 = (cnt + 7) >> 3;
#pragma unroll 1
            for (int it = 0; it < n8; ++it) {
                const float4 p0 = scratch4[4 * it], p1 = scratch4[4 * it + 1], p2 = scratch4[4 * it + 2], p3 = scratch4[4 * it + 3];
                acc0 += ex2_approx(fmaf(xgp, p0.x, p0.y));
                acc1 += ex2_approx(fmaf(xgp, p0.z, p0.w));
                acc2 += ex2_approx(fmaf(xgp, p1.x, p1.y));
                acc3 += ex2_approx(fmaf(xgp, p1.z, p1.w));
                acc0 += ex2_approx(fmaf(xgp, p2.x, p2.y));
                acc1 += ex2_approx(fmaf(xgp, p2.z, p2.w));
                acc2 += ex2_approx(fmaf(xgp, p3.x, p3.y));
                acc3 += ex2_approx(fmaf(xgp, p3.z, p3.w));
            }
            acc = ((acc0 + acc1) + (acc2 + acc3)) * ex2_approx(-xgp * xgp);
            __syncwarp();              // the scratch is rewritten by the next item
        } else {
            float acc0 = 0.f, acc1 = 0.f;
            int j = jb;
            for (; j + 2 <= je; j += 2) {
                const float2 s0_ = pk[j], s1_ = pk[j + 1];
                const float d0 = xg - s0_.x, d1 = xg - s1_.x;
                acc0 += ex2_approx(fmaf(-d0, d0, s0_.y));
                acc1 += ex2_approx(fmaf(-d1, d1, s1_.y));
            }
            if (j < je) {
                const float2 s0_ = pk[j];
                const float d0 = xg - s0_.x;
                acc0 += ex2_approx(fmaf(-d0, d0, s0_.y));
            }
            acc = acc0 + acc1;
        }
        if (valid) {
            double accd = (double)acc;
            double q = q_g[g];
            if (P.placement == CHIM_ON_GRID)
                q *= grid_factor(L, P.dc_tab + (size_t)l * (P.n_table + 1 + kZPad), P.n_table + 1 + kZPad,
                                 P.z_table_max / P.n_table, zc_g[g] + z0);
            lsum = fma(accd, q, lsum);
            if (P.dbg_K) atomicAdd(P.dbg_K + g, accd);
        }
    }
    const double knorm = (sw / ns) / ((double)ns * h * 2.50662827463100050242);
    double tot[1] = {lsum};
    block_sum<kEvThreads, 1>(tot, S.red);
    {
        double pr[1] = {(double)pairs};
        block_sum<kEvThreads, 1>(pr, S.red);
        if (tid == 0 && pr[0] > 0.0) atomicAdd(P.stats, (unsigned long long)pr[0]);
    }
    if (P.dbg_K) {   // diagnostics: turn the accumulated sums into K(z_g)
        __syncthreads();
        const double ks = knorm * exp(P.ln_shift[ev]);
        for (int g = tid; g < nz; g += kEvThreads) P.dbg_K[g] *= ks;
    }
    if (tid == 0) {
        double I = tot[0] * knorm;
        if (I > 0.0) *out = log(I) + P.ln_shift[ev];
        else if (I == 0.0) { *out = -INFINITY; atomicOr(P.flags + l, CHIM_FLAG_EVENT_ZERO); }
        else *out = NAN;
    }
}

size_t events_smem_bytes(int max_ns, int max_nz) {
    size_t ns_pad = ((size_t)max_ns + 3) & ~(size_t)3, max_tiles = ((size_t)max_nz + 31) / 32;
    return ((sizeof(EvSmem) + 15) / 16) * 16 + sizeof(double) * ns_pad + sizeof(float) * ev_float_region(ns_pad) +
           sizeof(int) * (3 * max_tiles + 1);
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
