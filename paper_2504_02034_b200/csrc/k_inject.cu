// k_inject.cu -- step S5 (selection term, eq. 12-13) and step S6 (combine, eq. 3).
//
//   S5  one CTA per (lambda, chunk of detected injections).  The lambda's mass table ("a" variant, 64 KB) is staged
//       once in shared memory -- the injections' source masses are scattered over the whole table, and scattered
//       16-byte reads cost an L1 wavefront each from global memory but ~1/3 of that from shared memory -- and the
//       chunk's packed records are streamed through it with coalesced 128-bit loads (the set is sorted in d_L, so a
//       warp's rows of the z(ln d_L) table are one or two cache lines).  CTAs in flight share a chunk (lambda is the
//       fast grid index), so the records come from L2.  Per (injection, lambda): s_j = p_m psi u / J / p_draw via the
//       same sample_weight() as the events (the injection table's R column carries psi u / J); z_j > z_cat_max gives
//       s_j = 0 (R6).  Per-CTA fp64 partial sums {sum s, sum s^2}, combined in a fixed order by S6 (deterministic).
//   S6  log L = sum_i log I_i - N_e log xi, N_eff (eq. 13), flags.
#include "chim_internal.cuh"

namespace chim {

constexpr int kInjThreads = 256;

struct InjSmem {
    LamConst L;
    double red[2 * (kInjThreads / 32)];
};

__global__ void __launch_bounds__(kInjThreads, 3) k_inject(InjKernelParams P) {
    extern __shared__ __align__(16) unsigned char smem_raw[];
    InjSmem& S = *reinterpret_cast<InjSmem*>(smem_raw);
    double2* sA = reinterpret_cast<double2*>(smem_raw + ((sizeof(InjSmem) + 15) / 16) * 16);
    double2* sB = sA + (P.n_mass + 2);
    const int tid = threadIdx.x, lane = tid & 31, wid = tid >> 5;
    const int l = blockIdx.x % P.n_lambda, chunk = blockIdx.x / P.n_lambda;
    const int64_t j0 = (int64_t)chunk * P.chunk, j1 = min(j0 + (int64_t)P.chunk, P.inj.n_det);
    const int nw = sizeof(LamConst) / 4;
    for (int i = tid; i < nw; i += kInjThreads)
        reinterpret_cast<uint32_t*>(&S.L)[i] = reinterpret_cast<const uint32_t*>(P.Lc + l)[i];
    MassLookup M;
    M.g = P.mtab + (size_t)l * (P.n_mass + 2);
    M.sA = sA; M.sB = sB; M.lo = 0; M.cap = P.n_mass + 2; M.n_mass = P.n_mass;
    for (int r = tid; r < P.n_mass + 2; r += kInjThreads) {
        double2 hi;
        const double2 lo = ldg256_lo(reinterpret_cast<const double*>(M.g + r), hi);
        sA[r] = lo;
        sB[r] = hi;
    }
    __syncthreads();
    const LamConst& L = S.L;
    double acc[2] = {0.0, 0.0};
    int oor = 0;
    if (L.flags == 0) {
        const Row* tab = P.tab + (size_t)l * P.tab_rows;
        // software pipeline: next sample's table coordinate one iteration ahead, its row prefetched to L1
        double2 A = (j0 + tid < j1) ? ldg_stream(P.inj.recA + j0 + tid) : make_double2(1.0, 1.0);
#pragma unroll 1
        for (int64_t j = j0 + tid; j < j1; j += kInjThreads) {
            const double2 B = ldg_stream(P.inj.recB + j), C = ldg_stream(P.inj.recC + j);
            double2 An = A;
            if (j + kInjThreads < j1) {
                An = ldg_stream(P.inj.recA + j + kInjThreads);
                prefetch_l1(tab + max(1, min((int)An.x, P.tab_rows - 2)));
            }
            double z, s;
            bool o;
            sample_weight(L, tab, P.tab_rows, M, L.tkmax_inj, P.z_table_max, A.x, A.y, B.x, B.y, C.x, C.y, z, s, o);
            oor |= (int)o;
            if (!(z <= P.z_cat_max)) s = 0.0;   // support of the selection-term z density (R6)
            acc[0] += s;
            acc[1] = fma(s, s, acc[1]);
            if (P.dbg_s) P.dbg_s[P.inj.perm[j]] = s * P.dbg_scale;
            A = An;
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
        P.partial[(size_t)chunk * P.n_lambda + l] = make_double2(a, b);
        if (oor) atomicOr(P.flags + l, CHIM_FLAG_TABLE_RANGE);
    }
}

size_t inject_smem_bytes(int n_mass) {
    return ((sizeof(InjSmem) + 15) / 16) * 16 + 2 * sizeof(double2) * (size_t)(n_mass + 2);
}

cudaError_t launch_inject(const InjKernelParams& P, int n_blocks, cudaStream_t st) {
    if (n_blocks <= 0) return cudaSuccess;
    size_t smem = inject_smem_bytes(P.n_mass);
    cudaError_t e = cudaFuncSetAttribute(k_inject, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    if (e != cudaSuccess) return e;
    k_inject<<<(unsigned)((long long)n_blocks * P.n_lambda), kInjThreads, smem, st>>>(P);
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
    double total = n_nan ? NAN : (n_ninf ? -INFINITY : v[0]);
    double logxi = 0.0, neff = NAN;
    if (lflags) { total = NAN; logxi = NAN; }
    else if (P.n_det > 0) {
        double xi = v[1] / P.n_inj_total;
        neff = v[1] * v[1] / (v[2] - v[1] * v[1] / P.n_inj_total);
        if (!(xi > 0.0)) { fl |= CHIM_FLAG_XI_ZERO; logxi = NAN; total = NAN; }
        else {
            logxi = log(xi) + P.inj_ln_shift;
            if (neff < P.neff_factor * P.n_events) fl |= CHIM_FLAG_NEFF_LOW;   // R8: report only
            total -= P.n_events * logxi;
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
