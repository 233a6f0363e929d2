// k_inject.cu -- step S5 (selection term, eq. 12-13) and step S6 (combine, eq. 3).
//
//   S5  one CTA per chunk of detected injections; the chunk's packed records are staged once in shared
//       memory and re-used for every lambda of the pass (so the injection set is streamed from HBM once per
//       pass, not once per lambda).  Per (injection, lambda): s_j = p_m psi u / J / p_draw via the same
//       sample_weight() as the events (the injection table's R column carries psi u / J); z_j > z_cat_max
//       gives s_j = 0 (R6).  Per-CTA fp64 partial sums {sum s, sum s^2} per lambda, combined in a fixed
//       order by S6 (deterministic; no atomics on the sums).
//   S6  log L = sum_i log I_i - N_e log xi, N_eff (eq. 13), flags.
#include "chim_internal.cuh"

namespace chim {

constexpr int kInjThreads = 256;

__device__ __forceinline__ void prefetch_l1(const void* p) { asm volatile("prefetch.global.L1 [%0];" ::"l"(p)); }

struct InjSmem {
    LamConst L[2];
    double red[2 * (kInjThreads / 32)];
};

__global__ void __launch_bounds__(kInjThreads) k_inject(InjKernelParams P) {
    extern __shared__ __align__(16) unsigned char smem_raw[];
    InjSmem& S = *reinterpret_cast<InjSmem*>(smem_raw);
    double2* rA = reinterpret_cast<double2*>(smem_raw + ((sizeof(InjSmem) + 15) / 16) * 16);
    double2* rB = rA + P.chunk;
    double2* rC = rB + P.chunk;
    const int tid = threadIdx.x, lane = tid & 31, wid = tid >> 5;
    const int64_t j0 = (int64_t)blockIdx.x * P.chunk;
    const int nj = (int)min((int64_t)P.chunk, P.inj.n_det - j0);
    for (int j = tid; j < nj; j += kInjThreads) {
        rA[j] = P.inj.recA[j0 + j];
        rB[j] = P.inj.recB[j0 + j];
        rC[j] = P.inj.recC[j0 + j];
    }
    const int nw = sizeof(LamConst) / 4;
    for (int i = tid; i < nw; i += kInjThreads)
        reinterpret_cast<uint32_t*>(&S.L[0])[i] = reinterpret_cast<const uint32_t*>(P.Lc)[i];
    __syncthreads();
    // the chunk is sorted in d_L, so it addresses the table rows [k_first, k_last] of every lambda's table
    const int k_first = max(1, (int)rA[0].x), k_span = min(P.tab_rows - 2, (int)rA[nj - 1].x) - k_first + 1;
    const int rho_lines = (P.n_win + 1 + 15) / 16;

    for (int l = 0; l < P.n_lambda; ++l) {
        const LamConst& L = S.L[l & 1];
        if (l + 1 < P.n_lambda) {   // prefetch the next lambda's constants (shared memory) and table lines (L1)
            for (int i = tid; i < nw; i += kInjThreads)
                reinterpret_cast<uint32_t*>(&S.L[(l + 1) & 1])[i] = reinterpret_cast<const uint32_t*>(P.Lc + l + 1)[i];
            if (tid < k_span) prefetch_l1(P.tab + (size_t)(l + 1) * P.tab_rows + k_first + tid);
            else if (tid - k_span < rho_lines) prefetch_l1(P.wtab + (size_t)(l + 1) * (P.n_win + 1) + 16 * (tid - k_span));
        }
        double acc[2] = {0.0, 0.0};
        int oor = 0;
        if (L.flags == 0) {
            const Row* tab = P.tab + (size_t)l * P.tab_rows;
            const double* wtab = P.wtab + (size_t)l * (P.n_win + 1);
#pragma unroll 1
            for (int j = tid; j < nj; j += kInjThreads) {
                double2 A = rA[j], B = rB[j], C = rC[j];
                double z, s;
                bool o;
                sample_weight(L, tab, P.tab_rows, wtab, P.n_win, L.tkmax_inj, P.z_table_max, A.x, A.y, B.x, B.y, C.x,
                              C.y, z, s, o);
                oor |= (int)o;
                if (!(z <= P.z_cat_max)) s = 0.0;   // support of the selection-term z density (R6)
                acc[0] += s;
                acc[1] += s * s;
                if (P.dbg_s) P.dbg_s[P.inj.perm[j0 + j]] = s * P.dbg_scale;
            }
        }
        acc[0] = warp_sum(acc[0]);
        acc[1] = warp_sum(acc[1]);
        if (lane == 0) { S.red[wid] = acc[0]; S.red[kInjThreads / 32 + wid] = acc[1]; }
        oor = __syncthreads_or(oor);   // also publishes S.red and the prefetched constants
        if (tid == 0) {
            double a = 0.0, b = 0.0;
#pragma unroll
            for (int k = 0; k < kInjThreads / 32; ++k) { a += S.red[k]; b += S.red[kInjThreads / 32 + k]; }
            P.partial[(size_t)blockIdx.x * P.n_lambda + l] = make_double2(a, b);
            if (oor) atomicOr(P.flags + l, CHIM_FLAG_TABLE_RANGE);
        }
        __syncthreads();   // S.red is re-used by the next lambda
    }
}

cudaError_t launch_inject(const InjKernelParams& P, int n_blocks, cudaStream_t st) {
    if (n_blocks <= 0) return cudaSuccess;
    size_t smem = ((sizeof(InjSmem) + 15) / 16) * 16 + 3 * sizeof(double2) * (size_t)P.chunk;
    cudaError_t e = cudaFuncSetAttribute(k_inject, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    if (e != cudaSuccess) return e;
    k_inject<<<n_blocks, kInjThreads, smem, st>>>(P);
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
