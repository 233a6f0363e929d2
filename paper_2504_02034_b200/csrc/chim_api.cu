// chim_api.cu -- the C ABI of libchim (include/chim.h): context, init-time packing, batch driver.
//
// Init (one-off, not on the hot path; SURVEY call stack (iii)): validate -> sort each event's samples by d_L
// (lambda-independent order: d_L^gw(z) is monotone, so sorted d_L means sorted z_j for every lambda) ->
// per-sample table coordinate in ln d_L, logs and mass ratio (all lambda-independent) -> centred grid and
// q_g = p_gal x trapezoid weight -> upload.  The batch call only enqueues kernels on the caller's stream.
#include <algorithm>
#include <cmath>
#include <cstdio>
#include <cstring>
#include <new>
#include <numeric>
#include <string>
#include <vector>

#include "chim_internal.cuh"

using namespace chim;

namespace {
constexpr size_t kMaxSmemOptin = 232448;   // 227 KB per CTA on sm_100
constexpr int kInjChunk = 16384;           // injections per CTA of k_inject (8192: +5 % time; 32768: same)
constexpr double kPolyMaxHalfRange = 0.45; // half-width in ln d_L up to which an event takes the local polynomials
}

struct chim_ctx {
    chim_config cfg;
    cudaStream_t stream = nullptr;
    std::string err;
    std::vector<void*> owned_ev, owned_inj, owned_work, owned_host, owned_ctx, owned_grp;
    int n_groups = 0;                      // many-1d grouping of the sub-events (0 = none)
    const int64_t* grp_off = nullptr; const double* grp_lnf = nullptr;
    const double* poly_mats = nullptr;     // fit matrices of the local polynomials (device)
    // events
    bool have_events = false;
    EventSetDev ev{};
    DlGrid ev_grid{0, 1, 0};
    const double* ev_ln_shift = nullptr;   // [n_events] added back to log I (prior scale factored out)
    const double* ev_ln_qscale = nullptr;  // [n_events] added back to log I (q_g scale factored out)
    std::vector<int64_t> h_sample_off, h_grid_off;
    // injections
    bool have_inj = false;
    InjSetDev inj{};
    DlGrid inj_grid{0, 1, 0};
    double inj_ln_shift = 0.0;
    int inj_blocks = 0;
    // work buffers for one lambda chunk
    int work_nl = 0;
    bool work_has_dc = false;
    LamConst* Lc = nullptr; Row* tab_ev = nullptr; Row* tab_inj = nullptr; MassRow* mtab = nullptr;
    double ev_m_top = 0.0, inj_m_top = 0.0;   // largest detector-frame m1 of each loaded set
    double* dc_tab = nullptr; double* logI = nullptr; double2* partial = nullptr; uint32_t* flags = nullptr;
    unsigned long long* stats = nullptr;
    float* poly_ev = nullptr; float* poly_inj = nullptr;   // local polynomials per (lambda, event) / (lambda, chunk)
    // S1 of the next lambda chunk runs on a stream of its own while S2-S6 of the current one fill the SMs (k_tables / k_polyfit
    // are latency-bound: few CTAs, many barriers): two sets of the S1 outputs, the pointers above name the set in use
    struct S1Set { LamConst* Lc; Row* tab_ev; Row* tab_inj; MassRow* mtab; double* dc_tab; float* poly_ev; float* poly_inj; };
    S1Set s1[2] = {};
    cudaStream_t aux_stream = nullptr;
    cudaEvent_t ev_begin = nullptr, ev_s1[2] = {nullptr, nullptr}, ev_rest[2] = {nullptr, nullptr};
    // k_events_fast: the events it takes / leaves to k_events, and the per-chunk work list of the units it hands over
    const int32_t* fast_ev = nullptr; const int32_t* slow_ev = nullptr;
    int n_fast = 0, n_slow = 0;
    int n_fast_c[kFastClasses] = {}, max_ns_c[kFastClasses] = {};   // the classes of k_events_fast (2 / 4 / 8 warps): events, longest sample list
    uint32_t* worklist = nullptr; unsigned int* work_count = nullptr;
    // staging for the host-pointer entry point
    int host_nl = 0;
    double* st_lam = nullptr; double* st_ll = nullptr; double* st_ev = nullptr; double* st_xi = nullptr;
    double* st_neff = nullptr; uint32_t* st_fl = nullptr;
    // chim_loglike_grad_batch: the displaced lambda rows and their results
    int grad_nl = 0;
    double* g_lam = nullptr; double* g_ll = nullptr; uint32_t* g_fl = nullptr;
    std::vector<void*> owned_grad;
    chim_stats last{};
    uint64_t launches = 0;
    // optional per-kernel timing (CUDA events around each launch of the last batch)
    bool profiling = false;
    int sm_count = 148;
    std::vector<cudaEvent_t> ev_pool;          // reused across batches
    std::vector<int> ev_kind;                  // kind of the launch bracketed by events [2i, 2i+1]
};

namespace {

thread_local std::string g_create_err;     // reason of the last failed chim_create on this thread: chim_last_error(NULL)
int fail(chim_ctx* c, int code, const std::string& msg) {
    if (c) c->err = msg;
    else g_create_err = msg;
    return code;
}
int cuda_fail(chim_ctx* c, cudaError_t e, const char* where) {
    return fail(c, e == cudaErrorMemoryAllocation ? CHIM_ENOMEM : CHIM_ECUDA,
                std::string(where) + ": " + cudaGetErrorString(e));
}
#define CK(call)                                                  \
    do {                                                          \
        cudaError_t e__ = (call);                                 \
        if (e__ != cudaSuccess) return cuda_fail(ctx, e__, #call); \
    } while (0)

template <class T>
cudaError_t dev_alloc(std::vector<void*>& pool, T** p, size_t n) {
    void* q = nullptr;
    cudaError_t e = cudaMalloc(&q, std::max<size_t>(n, 1) * sizeof(T));
    if (e == cudaSuccess) { pool.push_back(q); *p = static_cast<T*>(q); }
    return e;
}
void free_pool(std::vector<void*>& pool) {
    for (void* p : pool) cudaFree(p);
    pool.clear();
}
template <class T>
cudaError_t upload(std::vector<void*>& pool, const T** dst, const std::vector<T>& src) {
    T* d = nullptr;
    cudaError_t e = dev_alloc(pool, &d, src.size());
    if (e != cudaSuccess) return e;
    if (!src.empty()) e = cudaMemcpy(d, src.data(), src.size() * sizeof(T), cudaMemcpyHostToDevice);
    *dst = d;
    return e;
}
// bring an init input to the host (inputs live where cfg.mem says)
template <class T>
cudaError_t fetch(const chim_ctx* c, const T* src, size_t n, std::vector<T>& dst) {
    dst.resize(n);
    if (n == 0) return cudaSuccess;
    if (c->cfg.mem == CHIM_MEM_DEVICE) return cudaMemcpy(dst.data(), src, n * sizeof(T), cudaMemcpyDeviceToHost);
    std::memcpy(dst.data(), src, n * sizeof(T));
    return cudaSuccess;
}

// number of intervals of a z(ln d_L) table: the configured one, or (n_dl_table = 0) a spacing of ~0.005 in ln d_L,
// which keeps the interpolation error of the fp32 rows below their rounding
int choose_dl_intervals(const chim_ctx* ctx, double xmin, double xmax) {
    if (ctx->cfg.n_dl_table > 0) return std::min(ctx->cfg.n_dl_table, kMaxDlRows);
    double k = std::ceil((xmax - xmin) / 0.005);
    return (int)std::min<double>(std::max<double>(k, 64.0), (double)kMaxDlRows);
}

inline float f_hi(double x) { return (float)x; }
inline float f_lo(double x) { return (float)(x - (double)(float)x); }
inline float bits_f(uint32_t u) { float f; std::memcpy(&f, &u, 4); return f; }
inline uint32_t f_bits(float f) { uint32_t u; std::memcpy(&u, &f, 4); return u; }

DlGrid make_dl_grid(double xmin, double xmax, int K) {
    DlGrid g;
    g.x0 = xmin;
    g.K = K;
    double span = xmax - xmin;
    g.dx = (span > 0.0) ? span * (1.0 + 1e-12) / K + 1e-300 : 1e-6;
    return g;
}

// Work and host-staging buffers are sized for the loaded sets: dropped (and every pointer into them nulled) whenever a
// set is replaced.
void drop_work(chim_ctx* ctx) {
    free_pool(ctx->owned_work);
    ctx->work_nl = 0;
    ctx->work_has_dc = false;
    ctx->Lc = nullptr; ctx->tab_ev = nullptr; ctx->tab_inj = nullptr; ctx->mtab = nullptr; ctx->dc_tab = nullptr;
    ctx->logI = nullptr; ctx->partial = nullptr; ctx->flags = nullptr; ctx->stats = nullptr;
    ctx->poly_ev = nullptr; ctx->poly_inj = nullptr;
    ctx->s1[0] = chim_ctx::S1Set{}; ctx->s1[1] = chim_ctx::S1Set{};
    ctx->worklist = nullptr; ctx->work_count = nullptr;
    free_pool(ctx->owned_host);
    ctx->host_nl = 0;
    ctx->st_lam = ctx->st_ll = ctx->st_ev = ctx->st_xi = ctx->st_neff = nullptr;
    ctx->st_fl = nullptr;
}

int ensure_work(chim_ctx* ctx, int nl) {
    bool need_dc = ctx->cfg.placement == CHIM_ON_GRID;
    if (nl <= ctx->work_nl && (!need_dc || ctx->work_has_dc)) return CHIM_OK;
    {   // (the host staging is sized by n_lambda x n_events as well, but only grows with n_lambda: keep it)
        std::vector<void*> keep;
        keep.swap(ctx->owned_host);
        const int keep_nl = ctx->host_nl;
        double *a = ctx->st_lam, *b = ctx->st_ll, *c = ctx->st_ev, *d = ctx->st_xi, *e = ctx->st_neff;
        uint32_t* f = ctx->st_fl;
        drop_work(ctx);
        ctx->owned_host.swap(keep);
        ctx->host_nl = keep_nl;
        ctx->st_lam = a; ctx->st_ll = b; ctx->st_ev = c; ctx->st_xi = d; ctx->st_neff = e; ctx->st_fl = f;
    }
    CK(dev_alloc(ctx->owned_work, &ctx->Lc, nl));
    CK(dev_alloc(ctx->owned_work, &ctx->tab_ev, (size_t)nl * ctx->ev_grid.rows()));
    CK(dev_alloc(ctx->owned_work, &ctx->tab_inj, (size_t)nl * (ctx->have_inj ? ctx->inj_grid.rows() : 1)));
    CK(dev_alloc(ctx->owned_work, &ctx->mtab, (size_t)nl * 2 * (ctx->cfg.n_mass_table + 2)));
    ctx->dc_tab = nullptr;
    if (need_dc) CK(dev_alloc(ctx->owned_work, &ctx->dc_tab, (size_t)nl * (ctx->cfg.n_table + 1 + kZPad)));
    CK(dev_alloc(ctx->owned_work, &ctx->logI, (size_t)nl * ctx->ev.n_events));
    CK(dev_alloc(ctx->owned_work, &ctx->partial, (size_t)nl * std::max(ctx->inj_blocks, 1)));
    CK(dev_alloc(ctx->owned_work, &ctx->flags, nl));
    CK(dev_alloc(ctx->owned_work, &ctx->stats, 4));
    CK(dev_alloc(ctx->owned_work, &ctx->poly_ev, (size_t)nl * ctx->ev.n_events * 4 * kPolyN));
    CK(dev_alloc(ctx->owned_work, &ctx->poly_inj, (size_t)nl * std::max(ctx->inj_blocks, 1) * 4 * kPolyN));
    CK(dev_alloc(ctx->owned_work, &ctx->worklist, (size_t)nl * ctx->ev.n_events));
    CK(dev_alloc(ctx->owned_work, &ctx->work_count, 4));
    ctx->s1[0] = chim_ctx::S1Set{ctx->Lc, ctx->tab_ev, ctx->tab_inj, ctx->mtab, ctx->dc_tab, ctx->poly_ev, ctx->poly_inj};
    {   // the second set of the S1 outputs
        chim_ctx::S1Set& B = ctx->s1[1];
        CK(dev_alloc(ctx->owned_work, &B.Lc, nl));
        CK(dev_alloc(ctx->owned_work, &B.tab_ev, (size_t)nl * ctx->ev_grid.rows()));
        CK(dev_alloc(ctx->owned_work, &B.tab_inj, (size_t)nl * (ctx->have_inj ? ctx->inj_grid.rows() : 1)));
        CK(dev_alloc(ctx->owned_work, &B.mtab, (size_t)nl * 2 * (ctx->cfg.n_mass_table + 2)));
        B.dc_tab = nullptr;
        if (need_dc) CK(dev_alloc(ctx->owned_work, &B.dc_tab, (size_t)nl * (ctx->cfg.n_table + 1 + kZPad)));
        CK(dev_alloc(ctx->owned_work, &B.poly_ev, (size_t)nl * ctx->ev.n_events * 4 * kPolyN));
        CK(dev_alloc(ctx->owned_work, &B.poly_inj, (size_t)nl * std::max(ctx->inj_blocks, 1) * 4 * kPolyN));
    }
    ctx->work_nl = nl;
    ctx->work_has_dc = need_dc;
    return CHIM_OK;
}

void use_s1_set(chim_ctx* ctx, int k) {
    const chim_ctx::S1Set& B = ctx->s1[k];
    ctx->Lc = B.Lc; ctx->tab_ev = B.tab_ev; ctx->tab_inj = B.tab_inj; ctx->mtab = B.mtab; ctx->dc_tab = B.dc_tab;
    ctx->poly_ev = B.poly_ev; ctx->poly_inj = B.poly_inj;
}

TableParams table_params(const chim_ctx* ctx) {
    TableParams P;
    P.z_table_max = ctx->cfg.z_table_max;
    P.z_cat_max = ctx->cfg.z_cat_max;
    P.n_table = ctx->cfg.n_table;
    P.n_win = ctx->cfg.n_win_table;
    P.n_mass = ctx->cfg.n_mass_table;
    P.ln_m_top = std::log(std::max(std::max(ctx->ev_m_top, ctx->have_inj ? ctx->inj_m_top : 0.0), 1e-3));
    P.placement = ctx->cfg.placement;
    P.ev = ctx->ev_grid;
    P.inj = ctx->have_inj ? ctx->inj_grid : DlGrid{0, 1, 0};
    return P;
}

EventKernelParams event_params(const chim_ctx* ctx, int nl) {
    EventKernelParams P{};
    P.ev = ctx->ev;
    P.Lc = ctx->Lc; P.tab = ctx->tab_ev; P.mtab = ctx->mtab; P.dc_tab = ctx->dc_tab;
    P.n_lambda = nl; P.tab_rows = ctx->ev_grid.rows(); P.n_mass = ctx->cfg.n_mass_table; P.n_table = ctx->cfg.n_table;
    P.placement = ctx->cfg.placement; P.bw_rule = ctx->cfg.bw_rule; P.kde_method = ctx->cfg.kde_method; P.kde_kernel = ctx->cfg.kde_kernel; P.n_bins = ctx->cfg.n_bins;
    P.z_table_max = ctx->cfg.z_table_max; P.cutoff = ctx->cfg.kde_cutoff;
    // fp32 weights leave ~2e-5 / sqrt(n_eff) in log I: 64 keeps an event below 3e-6; the pixels of many-1d enter the event through a
    // sum over pixels (a 600-sample pixel has n_eff ~ 100), so a lower bar keeps them on the fast sweep
    P.neff_min = ctx->n_groups > 0 ? 24.f : 64.f;
    P.logI = ctx->logI; P.flags = ctx->flags; P.stats = ctx->stats;
    P.ln_shift = ctx->ev_ln_shift;
    P.ln_qscale = ctx->ev_ln_qscale;
    P.poly = ctx->poly_ev;
    P.dbg_event = -1;
    return P;
}

// profiling brackets: record an event pair around a launch of kind k (0 tables, 1 k_events_fast, 2 inject, 3 combine, 4 k_events)
struct Bracket {
    chim_ctx* ctx; bool on; size_t slot;
    Bracket(chim_ctx* c, int kind) : ctx(c), on(c->profiling), slot(0) {
        if (!on) return;
        slot = ctx->ev_kind.size();
        while (ctx->ev_pool.size() < 2 * (slot + 1)) {
            cudaEvent_t e;
            if (cudaEventCreate(&e) != cudaSuccess) { on = false; return; }
            ctx->ev_pool.push_back(e);
        }
        ctx->ev_kind.push_back(kind);
        cudaEventRecord(ctx->ev_pool[2 * slot], ctx->stream);
    }
    ~Bracket() { if (on) cudaEventRecord(ctx->ev_pool[2 * slot + 1], ctx->stream); }
};

// S1 of one chunk of lambdas into the set of buffers in use, on stream `st` (timed only when it is the context's stream)
int run_s1(chim_ctx* ctx, int nl, const double* lam, cudaStream_t st) {
    TableParams TP = table_params(ctx);
    const bool timed = st == ctx->stream;
    const bool prof = ctx->profiling;
    if (!timed) ctx->profiling = false;
    int rc = [&]() -> int {
        { Bracket b(ctx, 0); CK(launch_tables(lam, nl, TP, ctx->Lc, ctx->dc_tab, ctx->tab_ev, ctx->tab_inj, ctx->mtab, st)); }
        {   // local-polynomial fits (part of S1: per-lambda interpolants)
            Bracket b(ctx, 0);
            CK(launch_polyfit(ctx->Lc, ctx->tab_ev, ctx->ev_grid.rows(), nl, ctx->ev.n_events, ctx->ev.tk_c, ctx->ev.tk_h, ctx->ev.z0, 0.0,
                              false, ctx->poly_mats, ctx->ev.lnm1_lo, ctx->ev.lnm1_hi, ctx->cfg.n_mass_table,
                              events_mass_stage_rows(ctx->cfg.n_mass_table), ctx->ev_grid.dx, ctx->poly_ev, st));
            if (ctx->have_inj)
                CK(launch_polyfit(ctx->Lc, ctx->tab_inj, ctx->inj_grid.rows(), nl, ctx->inj_blocks, ctx->inj.tk_c, ctx->inj.tk_h, nullptr,
                                  ctx->cfg.z_cat_max, true, ctx->poly_mats, nullptr, nullptr, 0, 0, ctx->inj_grid.dx, ctx->poly_inj, st));
            ctx->launches += ctx->have_inj ? 2 : 1;
        }
        ctx->launches += 1;   // (k_tables)
        return CHIM_OK;
    }();
    ctx->profiling = prof;
    return rc;
}

// S2-S4 -> S5 -> S6 of one chunk on the context's stream, from the set of S1 outputs in use
int run_rest(chim_ctx* ctx, int nl, double* out_ll, double* out_ev, double* out_xi, double* out_neff, uint32_t* out_fl) {
    cudaStream_t st = ctx->stream;
    CK(cudaMemsetAsync(ctx->flags, 0, sizeof(uint32_t) * nl, st));
    EventKernelParams EP = event_params(ctx, nl);
    const chim_config& cf = ctx->cfg;
    // the regular units go to k_events_fast: default configuration (Gaussian kernel, local-expansion form, weights on the samples,
    // no binning, no pair counting) and events with a narrow d_L range on an equally spaced grid; the rest, and every unit the
    // fast kernel hands over through the work list, to k_events
    const bool fast = ctx->n_fast > 0 && cf.placement == CHIM_ON_SAMPLES && cf.kde_kernel == CHIM_KERNEL_GAUSS && cf.n_bins == 0 &&
                      cf.kde_method == CHIM_KDE_AUTO && cf.kde_cutoff > 0.0 && cf.count_pairs == 0;
    if (fast) {
        FastEventParams FP{};
        FP.ev = ctx->ev; FP.Lc = ctx->Lc; FP.mtab = ctx->mtab; FP.poly = ctx->poly_ev;
        FP.n_lambda = nl; FP.n_mass = cf.n_mass_table; FP.bw_rule = cf.bw_rule; FP.cutoff = cf.kde_cutoff; FP.neff_min = EP.neff_min;
        FP.logI = ctx->logI; FP.ln_shift = ctx->ev_ln_shift; FP.ln_qscale = ctx->ev_ln_qscale;
        FP.fast_events = ctx->fast_ev; FP.worklist = ctx->worklist; FP.work_count = ctx->work_count;
        CK(cudaMemsetAsync(ctx->work_count, 0, sizeof(unsigned int), st));
        for (int c = 0, first = 0; c < kFastClasses; first += ctx->n_fast_c[c], ++c) {
            if (ctx->n_fast_c[c] == 0) continue;
            FP.fast_events = ctx->fast_ev + first;
            FP.warps = 2 << c; FP.max_d = fast_max_d_for(FP.warps, ctx->ev.max_nz); FP.max_ns = ctx->max_ns_c[c];
            { Bracket b(ctx, 1); CK(launch_events_fast(FP, ctx->n_fast_c[c], st)); }
            ctx->launches += 1;
        }
        if (ctx->n_slow > 0) {
            EP.ev_list = ctx->slow_ev; EP.n_ev_list = ctx->n_slow;
            { Bracket b(ctx, 4); CK(launch_events(EP, false, st)); }
            ctx->launches += 1;
        }
        EP.ev_list = nullptr; EP.n_ev_list = 0;
        EP.worklist = ctx->worklist; EP.work_count = ctx->work_count;
        EP.worklist_ctas = (int)std::min<long long>((long long)nl * ctx->n_fast, 3LL * ctx->sm_count);
        { Bracket b(ctx, 4); CK(launch_events(EP, false, st)); }
        ctx->launches += 1;
    } else {
        { Bracket b(ctx, 4); CK(launch_events(EP, cf.count_pairs != 0, st)); }
        ctx->launches += 1;
    }
    if (ctx->have_inj) {
        InjKernelParams IP{};
        IP.inj = ctx->inj; IP.Lc = ctx->Lc; IP.tab = ctx->tab_inj; IP.mtab = ctx->mtab;
        IP.n_lambda = nl; IP.tab_rows = ctx->inj_grid.rows(); IP.n_mass = ctx->cfg.n_mass_table; IP.chunk = kInjChunk;
        IP.z_table_max = ctx->cfg.z_table_max; IP.z_cat_max = ctx->cfg.z_cat_max;
        IP.partial = ctx->partial; IP.flags = ctx->flags; IP.dbg_s = nullptr; IP.poly = ctx->poly_inj; IP.n_chunks = ctx->inj_blocks;
        { Bracket b(ctx, 2); CK(launch_inject(IP, ctx->inj_blocks, st)); }
        ctx->launches += 1;
    }
    CombineParams CP{};
    CP.Lc = ctx->Lc; CP.logI = ctx->logI; CP.partial = ctx->partial;
    CP.n_lambda = nl; CP.n_events = ctx->ev.n_events; CP.n_inj_blocks = ctx->inj_blocks;
    CP.n_det = ctx->have_inj ? ctx->inj.n_det : 0;
    CP.n_inj_total = ctx->have_inj ? ctx->inj.n_inj_total : 1.0;
    CP.inj_ln_shift = ctx->inj_ln_shift;
    CP.n_groups = ctx->n_groups; CP.group_off = ctx->grp_off; CP.ln_factor = ctx->grp_lnf;
    CP.neff_factor = ctx->cfg.neff_factor; CP.flags_in = ctx->flags;
    CP.out_loglike = out_ll; CP.out_event_logI = out_ev; CP.out_logxi = out_xi; CP.out_neff = out_neff; CP.out_flags = out_fl;
    { Bracket b(ctx, 3); CK(launch_combine(CP, st)); }
    ctx->launches += 1;
    return CHIM_OK;
}

// Chebyshev nodes and the node-value -> monomial-coefficient matrices of the local polynomials (chim_internal.cuh)
cudaError_t upload_poly_matrices(chim_ctx* ctx) {
    constexpr int N = kPolyN;
    std::vector<double> h(kPolyMatDoubles, 0.0);
    double A[N][N], C[N][N] = {};
    const double pi = 3.14159265358979323846;
    for (int k = 0; k < N; ++k) h[k] = std::cos(pi * (k + 0.5) / N);
    for (int m = 0; m < N; ++m)            // Chebyshev coefficient m from the node values (discrete orthogonality)
        for (int k = 0; k < N; ++k) A[m][k] = (m == 0 ? 1.0 : 2.0) / N * std::cos(m * pi * (k + 0.5) / N);
    C[0][0] = 1.0;                         // C[n][m]: coefficient of t^n in T_m
    C[1][1] = 1.0;
    for (int m = 2; m < N; ++m)
        for (int n = 0; n < N; ++n) C[n][m] = (n > 0 ? 2.0 * C[n - 1][m - 1] : 0.0) - C[n][m - 2];
    for (int n = 0; n < N; ++n)
        for (int k = 0; k < N; ++k) {
            double a7 = 0.0, a6 = 0.0;
            for (int m = 0; m < N; ++m) {
                a7 += C[n][m] * A[m][k];
                if (m < N - 1) a6 += C[n][m] * A[m][k];
            }
            h[N + n * N + k] = a7;
            h[N + N * N + n * N + k] = (n < N - 1) ? a6 : 0.0;
        }
    return upload(ctx->owned_ctx, &ctx->poly_mats, h);
}

bool all_finite(const std::vector<double>& v) {
    for (double x : v) if (!std::isfinite(x)) return false;
    return true;
}

}  // namespace

extern "C" {

void chim_default_config(chim_config* cfg) {
    if (!cfg) return;
    std::memset(cfg, 0, sizeof(*cfg));
    cfg->device = 0;
    cfg->mem = CHIM_MEM_HOST;
    cfg->stream = nullptr;
    cfg->placement = CHIM_ON_SAMPLES;
    cfg->bw_rule = CHIM_BW_SCOTT;
    cfg->kde_cutoff = 6.0;
    cfg->z_cat_max = 1.5;
    cfg->z_table_max = 10.0;
    cfg->n_table = 2048;
    cfg->n_dl_table = 0;
    cfg->n_win_table = 512;
    cfg->lambda_chunk = 1024;
    cfg->neff_factor = 5.0;
    cfg->kde_method = CHIM_KDE_AUTO;
    cfg->n_mass_table = 1024;
    cfg->count_pairs = 0;
    cfg->kde_kernel = CHIM_KERNEL_GAUSS;
    cfg->n_bins = 0;
}

int chim_version(void) { return CHIM_VERSION; }

#ifndef CHIM_BUILD_ID
#define CHIM_BUILD_ID "unknown"
#endif
const char* chim_build_id(void) { return CHIM_BUILD_ID; }

const char* chim_last_error(const chim_ctx* ctx) { return ctx ? ctx->err.c_str() : g_create_err.c_str(); }

int chim_create(const chim_config* cfg, chim_ctx** out) {
    if (!out) return fail(nullptr, CHIM_EINVAL, "chim_create: out is NULL");
    *out = nullptr;
    chim_config c;
    if (cfg) c = *cfg; else chim_default_config(&c);
    chim_config d;
    chim_default_config(&d);
    if (c.n_table <= 0) c.n_table = d.n_table;
    if (c.n_dl_table < 0) c.n_dl_table = d.n_dl_table;
    if (c.n_win_table <= 0) c.n_win_table = d.n_win_table;
    if (c.lambda_chunk <= 0) c.lambda_chunk = d.lambda_chunk;
    if (c.n_mass_table <= 0) c.n_mass_table = d.n_mass_table;
    if (!(c.z_table_max > 0.0)) c.z_table_max = d.z_table_max;
    if (!(c.z_cat_max > 0.0)) c.z_cat_max = d.z_cat_max;
    if (!(c.neff_factor >= 0.0)) c.neff_factor = d.neff_factor;
    if (c.kde_cutoff < 0.0 || !std::isfinite(c.kde_cutoff)) return fail(nullptr, CHIM_EINVAL, "chim_create: kde_cutoff must be finite and >= 0");
    if (c.n_table < 16 || (c.n_dl_table != 0 && c.n_dl_table < 16) || c.n_dl_table > kMaxDlRows || c.n_win_table < 8 || c.n_mass_table < 64)
        return fail(nullptr, CHIM_EINVAL, "chim_create: table size out of range (n_table >= 16, n_dl_table 0 or 16..4093, n_win_table >= 8, n_mass_table >= 64)");
    if (c.z_cat_max > c.z_table_max) return fail(nullptr, CHIM_EINVAL, "chim_create: z_cat_max exceeds z_table_max");
    if (c.placement != CHIM_ON_SAMPLES && c.placement != CHIM_ON_GRID) return fail(nullptr, CHIM_EINVAL, "chim_create: unknown placement");
    if (c.bw_rule != CHIM_BW_SCOTT && c.bw_rule != CHIM_BW_FIXED) return fail(nullptr, CHIM_EINVAL, "chim_create: unknown bw_rule");
    if (c.kde_method != CHIM_KDE_AUTO && c.kde_method != CHIM_KDE_DIRECT && c.kde_method != CHIM_KDE_POWER && c.kde_method != CHIM_KDE_NONE)
        return fail(nullptr, CHIM_EINVAL, "chim_create: unknown kde_method");
    if (c.mem != CHIM_MEM_HOST && c.mem != CHIM_MEM_DEVICE) return fail(nullptr, CHIM_EINVAL, "chim_create: unknown mem");
    if (c.kde_kernel != CHIM_KERNEL_GAUSS && c.kde_kernel != CHIM_KERNEL_EPANECHNIKOV) return fail(nullptr, CHIM_EINVAL, "chim_create: unknown kde_kernel");
    if (c.n_bins < 0 || c.n_bins > 2048) return fail(nullptr, CHIM_EINVAL, "chim_create: n_bins must be in [0, 2048]");
    if (c.kde_kernel == CHIM_KERNEL_EPANECHNIKOV && c.placement != CHIM_ON_SAMPLES)   // lambda-independent q_g needed
        return fail(nullptr, CHIM_EINVAL, "chim_create: the Epanechnikov kernel needs placement CHIM_ON_SAMPLES");
    int ndev = 0;
    cudaError_t ce = cudaGetDeviceCount(&ndev);
    if (ce != cudaSuccess) return fail(nullptr, CHIM_ECUDA, std::string("chim_create: cudaGetDeviceCount: ") + cudaGetErrorString(ce));
    if (c.device < 0 || c.device >= ndev) return fail(nullptr, CHIM_ECUDA, "chim_create: no such CUDA device");
    cudaDeviceProp prop;
    ce = cudaGetDeviceProperties(&prop, c.device);
    if (ce != cudaSuccess) return fail(nullptr, CHIM_ECUDA, std::string("chim_create: cudaGetDeviceProperties: ") + cudaGetErrorString(ce));
    if (prop.major != 10)   // sm_100a only: no other code path exists
        return fail(nullptr, CHIM_ECUDA, std::string("chim_create: device is ") + prop.name + " (compute capability " + std::to_string(prop.major) + "." +
                                         std::to_string(prop.minor) + "); libchim is built for sm_100a only");
    ce = cudaSetDevice(c.device);
    if (ce != cudaSuccess) return fail(nullptr, CHIM_ECUDA, std::string("chim_create: cudaSetDevice: ") + cudaGetErrorString(ce));
    chim_ctx* ctx = new (std::nothrow) chim_ctx();
    if (!ctx) return fail(nullptr, CHIM_ENOMEM, "chim_create: out of host memory");
    ctx->cfg = c;
    ctx->sm_count = prop.multiProcessorCount;
    ctx->stream = static_cast<cudaStream_t>(c.stream);
    TableParams TP = table_params(ctx);
    TP.ev.K = TP.inj.K = c.n_dl_table > 0 ? c.n_dl_table : kMaxDlRows;
    if (tables_smem_bytes(TP) > kMaxSmemOptin || inject_smem_bytes(c.n_mass_table) > kMaxSmemOptin) {
        delete ctx;
        return fail(nullptr, CHIM_EINVAL, "chim_create: n_table / n_win_table / n_mass_table exceed the shared-memory staging limit");
    }
    ce = upload_gauss_legendre();
    if (ce == cudaSuccess) ce = upload_poly_matrices(ctx);
    if (ce == cudaSuccess) {   // the auxiliary stream of S1 (highest priority: its few CTAs go ahead of the queued S2-S5 ones) and its events
        int pr_lo = 0, pr_hi = 0;
        cudaDeviceGetStreamPriorityRange(&pr_lo, &pr_hi);
        ce = cudaStreamCreateWithPriority(&ctx->aux_stream, cudaStreamNonBlocking, pr_hi);
        cudaEvent_t* evs[5] = {&ctx->ev_begin, &ctx->ev_s1[0], &ctx->ev_s1[1], &ctx->ev_rest[0], &ctx->ev_rest[1]};
        for (int i = 0; i < 5 && ce == cudaSuccess; ++i) ce = cudaEventCreateWithFlags(evs[i], cudaEventDisableTiming);
    }
    if (ce != cudaSuccess) {
        chim_destroy(ctx);
        return fail(nullptr, ce == cudaErrorMemoryAllocation ? CHIM_ENOMEM : CHIM_ECUDA, std::string("chim_create: ") + cudaGetErrorString(ce));
    }
    *out = ctx;
    return CHIM_OK;
}

void chim_destroy(chim_ctx* ctx) {
    if (!ctx) return;
    cudaSetDevice(ctx->cfg.device);
    cudaStreamSynchronize(ctx->stream);
    if (ctx->aux_stream) { cudaStreamSynchronize(ctx->aux_stream); cudaStreamDestroy(ctx->aux_stream); }
    for (cudaEvent_t e : {ctx->ev_begin, ctx->ev_s1[0], ctx->ev_s1[1], ctx->ev_rest[0], ctx->ev_rest[1]})
        if (e) cudaEventDestroy(e);
    for (cudaEvent_t e : ctx->ev_pool) cudaEventDestroy(e);
    free_pool(ctx->owned_ev);
    free_pool(ctx->owned_inj);
    free_pool(ctx->owned_work);
    free_pool(ctx->owned_host);
    free_pool(ctx->owned_ctx);
    free_pool(ctx->owned_grp);
    free_pool(ctx->owned_grad);
    delete ctx;
}

int chim_init_events(chim_ctx* ctx, int32_t n_events, const int64_t* sample_off, const double* dL, const double* m1d,
                     const double* m2d, const double* ln_prior, const int64_t* grid_off, const double* z_grid,
                     const double* p_gal, const double* fixed_bw) {
    if (!ctx) return CHIM_EINVAL;
    if (n_events < 1 || !sample_off || !dL || !m1d || !m2d || !ln_prior || !grid_off || !z_grid || !p_gal)
        return fail(ctx, CHIM_EINVAL, "chim_init_events: null pointer or n_events < 1");
    if (ctx->cfg.bw_rule == CHIM_BW_FIXED && !fixed_bw)
        return fail(ctx, CHIM_EINVAL, "chim_init_events: bw_rule is CHIM_BW_FIXED but fixed_bw is NULL");
    CK(cudaSetDevice(ctx->cfg.device));
    std::vector<int64_t> so, go;
    CK(fetch(ctx, sample_off, (size_t)n_events + 1, so));
    CK(fetch(ctx, grid_off, (size_t)n_events + 1, go));
    if (so[0] != 0 || go[0] != 0) return fail(ctx, CHIM_EINVAL, "chim_init_events: offsets must start at 0");
    int max_ns = 0, max_nz = 0;
    for (int i = 0; i < n_events; ++i) {
        int64_t ns = so[i + 1] - so[i], nz = go[i + 1] - go[i];
        if (ns < 1 || nz < 2 || ns > (1 << 30) || nz > (1 << 30))
            return fail(ctx, CHIM_EINVAL, "chim_init_events: every event needs N_s >= 1 samples and N_z >= 2 grid points");
        max_ns = std::max<int>(max_ns, (int)ns);
        max_nz = std::max<int>(max_nz, (int)nz);
    }
    if (ctx->cfg.n_bins > max_ns)
        return fail(ctx, CHIM_EINVAL, "chim_init_events: cfg.n_bins exceeds the largest N_s (the pseudo-samples reuse the sample stage)");
    if (events_smem_bytes(max_ns, max_nz) > kMaxSmemOptin) {
        char b[160];
        std::snprintf(b, sizeof b, "chim_init_events: N_s = %d exceeds the shared-memory staging limit (%d samples per event)",
                      max_ns, (int)((kMaxSmemOptin - 4096 - 8 * (size_t)max_nz) / 12));
        return fail(ctx, CHIM_EINVAL, b);
    }
    const size_t NS = (size_t)so[n_events], NG = (size_t)go[n_events];
    std::vector<double> h_dl, h_m1, h_m2, h_lp, h_z, h_p, h_bw;
    CK(fetch(ctx, dL, NS, h_dl)); CK(fetch(ctx, m1d, NS, h_m1)); CK(fetch(ctx, m2d, NS, h_m2));
    CK(fetch(ctx, ln_prior, NS, h_lp)); CK(fetch(ctx, z_grid, NG, h_z)); CK(fetch(ctx, p_gal, NG, h_p));
    if (fixed_bw) CK(fetch(ctx, fixed_bw, (size_t)n_events, h_bw));
    if (!all_finite(h_dl) || !all_finite(h_m1) || !all_finite(h_m2) || !all_finite(h_lp) || !all_finite(h_z) ||
        !all_finite(h_p) || !all_finite(h_bw))
        return fail(ctx, CHIM_EINVAL, "chim_init_events: non-finite input");
    double xmin = INFINITY, xmax = -INFINITY, m_top = 0.0;
    for (size_t j = 0; j < NS; ++j) {
        if (!(h_dl[j] > 0.0) || !(h_m2[j] > 0.0) || !(h_m1[j] >= h_m2[j]))
            return fail(ctx, CHIM_EINVAL, "chim_init_events: need dL > 0 and m1d >= m2d > 0");
        m_top = std::max(m_top, h_m1[j]);
        double x = std::log(h_dl[j]);
        xmin = std::min(xmin, x);
        xmax = std::max(xmax, x);
    }
    for (int i = 0; i < n_events; ++i) {
        for (int64_t g = go[i]; g < go[i + 1]; ++g) {
            if (h_z[g] < 0.0 || h_p[g] < 0.0 || (g > go[i] && !(h_z[g] > h_z[g - 1])))
                return fail(ctx, CHIM_EINVAL, "chim_init_events: z_grid must be >= 0 and strictly increasing, p_gal >= 0");
        }
        if (ctx->cfg.bw_rule == CHIM_BW_FIXED && !(h_bw[i] > 0.0))
            return fail(ctx, CHIM_EINVAL, "chim_init_events: fixed_bw must be > 0");
    }
    DlGrid grid = make_dl_grid(xmin, xmax, choose_dl_intervals(ctx, xmin, xmax));

    std::vector<float4> rec(2 * NS);
    // records of the event-local-polynomial sweep: {m1d, m2d, t, ln m1d}, {ln m2d, log2(1/prior) - scale, 0, 0}; every
    // event padded to a multiple of 32 samples with copies of its last one (whole warps read without bounds checks)
    std::vector<int64_t> poff(n_events + 1, 0);
    for (int i = 0; i < n_events; ++i) poff[i + 1] = poff[i] + ((so[i + 1] - so[i] + 31) / 32) * 32;
    constexpr size_t kRecTail = 1024;   // spare records: the sweeps prefetch one iteration (256 records) past their range
    std::vector<float4> prec_a((size_t)poff[n_events] + kRecTail, make_float4(1.f, 1.f, 0.f, 0.f));
    std::vector<float2> prec_b((size_t)poff[n_events] + kRecTail, make_float2(0.f, 0.f));
    std::vector<int32_t> k_lo(n_events), k_hi(n_events);
    const double l2e = 1.4426950408889634074;
    std::vector<int32_t> perm(NS);
    std::vector<double> zc(NG), qg(NG), z0(n_events), shift(n_events), qshift(n_events), udz(n_events), maxdz(n_events);
    std::vector<float> qn(NG);
    std::vector<double> ep0(NG + n_events), ep1(NG + n_events), ep2(NG + n_events);   // Epanechnikov prefix sums
    std::vector<double> lm_lo(n_events), lm_hi(n_events);
    std::vector<float2> chunk_top((size_t)n_events * kFastWarps, make_float2(0.f, 1.f));   // k_events_fast: per chunk {largest m2d, t of its last sample}
    std::vector<double> tk_c(n_events), tk_h(n_events);
    std::vector<uint32_t> tkq_c(n_events);
    std::vector<float> tq_scale(n_events);   // (host-side intermediates of the polynomial coordinate)
    std::vector<int32_t> idx;
    for (int i = 0; i < n_events; ++i) {
        const int64_t s0 = so[i];
        const int ns = (int)(so[i + 1] - s0);
        idx.resize(ns);
        std::iota(idx.begin(), idx.end(), 0);
        std::stable_sort(idx.begin(), idx.end(), [&](int a, int b) { return h_dl[s0 + a] < h_dl[s0 + b]; });
        double sh = -INFINITY;   // factor the prior scale out of the weights: 1/pi_j = exp(sh) * ipr_j
        for (int j = 0; j < ns; ++j) sh = std::max(sh, -h_lp[s0 + j]);
        shift[i] = sh;
        lm_lo[i] = INFINITY;
        lm_hi[i] = -INFINITY;
        for (int j = 0; j < ns; ++j) {
            const int64_t o = s0 + idx[j];
            lm_lo[i] = std::min(lm_lo[i], std::log(h_m1[o]));
            lm_hi[i] = std::max(lm_hi[i], std::log(h_m1[o]));
            const double tk = (std::log(h_dl[o]) - grid.x0) / grid.dx + 1.0;   // in [1, K + 1)
            const uint32_t tkq_max = ((uint32_t)(grid.K + 1) << kTkFracBits) - 1u;   // rounding must not leave the last interval
            const uint32_t tkq = std::min((uint32_t)std::min<double>(std::max(tk, 0.0) * (double)(1u << kTkFracBits) + 0.5, 4294967295.0), tkq_max);
            rec[2 * (s0 + j)] = make_float4(bits_f(tkq), f_hi(h_m1[o]), f_lo(h_m1[o]), f_hi(h_m2[o]));
            rec[2 * (s0 + j) + 1] = make_float4(f_lo(h_m2[o]), (float)std::log(h_m1[o]), (float)std::log(h_m2[o] / h_m1[o]),
                                     (float)(l2e * (-h_lp[o] - sh)));   // log2(1/pi_j) with the event's scale removed
            perm[s0 + j] = idx[j];
            const int k = std::min(std::max((int)(tkq >> kTkFracBits), 1), grid.K);
            if (j == 0) k_lo[i] = k;
            k_hi[i] = k;
        }
        {   // event-local polynomials of k_events: centre / half-width of the samples in table coordinates
            const double fq = (double)(1u << kTkFracBits);
            const double q_lo = (double)f_bits(rec[2 * s0].x), q_hi = (double)f_bits(rec[2 * (s0 + ns - 1)].x);
            tkq_c[i] = (uint32_t)(0.5 * (q_lo + q_hi));
            tk_c[i] = (double)tkq_c[i] / fq;
            const double half = std::max(q_hi - (double)tkq_c[i], (double)tkq_c[i] - q_lo) / fq + 1e-3;
            tk_h[i] = (half * grid.dx <= kPolyMaxHalfRange) ? half : 0.0;
            tq_scale[i] = (float)(1.0 / (half * fq));
            const int64_t p0 = poff[i], np = poff[i + 1] - p0;
            for (int64_t j = 0; j < np; ++j) {
                const int64_t js = s0 + std::min<int64_t>(j, ns - 1), o = s0 + idx[std::min<int64_t>(j, ns - 1)];
                const double t = ((double)f_bits(rec[2 * js].x) - (double)tkq_c[i]) / (half * fq);
                prec_a[p0 + j] = make_float4((float)h_m1[o], (float)h_m2[o], (float)t, (float)std::log(h_m1[o]));
                if (j < ns) {
                    float2& ct = chunk_top[(size_t)i * kFastWarps + std::min<int64_t>(j / fast_chunk((int)ns, fast_warps_for((int)ns)), fast_warps_for((int)ns) - 1)];
                    ct.x = std::max(ct.x, (float)h_m2[o]);
                    ct.y = (float)t;                                   // (samples in d_L order: the last one written is the chunk's last)
                }
                prec_b[p0 + j] = make_float2((float)std::log(h_m2[o]), rec[2 * js + 1].w);
            }
        }
        const int64_t g0 = go[i];
        const int nz = (int)(go[i + 1] - g0);
        z0[i] = 0.5 * (h_z[g0] + h_z[g0 + nz - 1]);
        for (int g = 0; g < nz; ++g) {
            double wl = (g > 0) ? h_z[g0 + g] - h_z[g0 + g - 1] : 0.0;
            double wr = (g + 1 < nz) ? h_z[g0 + g + 1] - h_z[g0 + g] : 0.0;
            zc[g0 + g] = h_z[g0 + g] - z0[i];
            qg[g0 + g] = h_p[g0 + g] * 0.5 * (wl + wr);   // composite trapezoid weight (O9)
        }
        // q_g normalised by the event's largest value (kept in fp32; the scale returns in log I)
        double qmax = 0.0;
        for (int g = 0; g < nz; ++g) qmax = std::max(qmax, qg[g0 + g]);
        if (!(qmax > 0.0)) qmax = 1.0;
        qshift[i] = std::log(qmax);
        for (int g = 0; g < nz; ++g) qn[g0 + g] = (float)(qg[g0 + g] / qmax);
        {
            long double a0 = 0.0L, a1 = 0.0L, a2 = 0.0L;
            const size_t e0 = (size_t)g0 + i;
            ep0[e0] = ep1[e0] = ep2[e0] = 0.0;
            for (int g = 0; g < nz; ++g) {
                const long double q = qg[g0 + g] / qmax, zz = zc[g0 + g];
                a0 += q; a1 += q * zz; a2 += q * zz * zz;
                ep0[e0 + g + 1] = (double)a0; ep1[e0 + g + 1] = (double)a1; ep2[e0 + g + 1] = (double)a2;
            }
        }
        // equally spaced grid?  then the KDE pair loop may take the power form
        const double dz = (h_z[g0 + nz - 1] - h_z[g0]) / (nz - 1);
        bool uniform = true;
        for (int g = 0; g < nz && uniform; ++g) uniform = std::fabs(h_z[g0 + g] - (h_z[g0] + g * dz)) <= 1e-7 * dz;
        udz[i] = uniform ? dz : 0.0;
        maxdz[i] = 0.0;
        for (int g = 1; g < nz; ++g) maxdz[i] = std::max(maxdz[i], h_z[g0 + g] - h_z[g0 + g - 1]);
    }
    // k_events_fast: q_g once more with 16-byte aligned, zero-padded slices (the source of its TMA copy), and the events it takes:
    // narrow d_L range (event-local polynomials) on an equally spaced grid, if its stage fits the shared memory at all
    std::vector<int64_t> q4off(n_events);
    int64_t q4n = 0;
    for (int i = 0; i < n_events; ++i) { q4off[i] = q4n; q4n += ((go[i + 1] - go[i] + 3) / 4) * 4; }
    std::vector<float> qn4((size_t)q4n + 4, 0.f);
    for (int i = 0; i < n_events; ++i) std::copy(qn.begin() + go[i], qn.begin() + go[i + 1], qn4.begin() + q4off[i]);
    // k_events_fast takes the events with a narrow d_L range on an equally spaced grid, in two classes by the length of the
    // sample list (chim_internal.cuh: fast_warps_for), the classes one after the other in the list
    std::vector<int32_t> fast_ev, slow_ev;
    int n_fast_c[kFastClasses] = {}, max_ns_c[kFastClasses] = {};
    for (int c = 0; c < kFastClasses; ++c) {
        const int w = 2 << c;
        for (int i = 0; i < n_events; ++i)
            if (fast_warps_for((int)(so[i + 1] - so[i])) == w) max_ns_c[c] = std::max(max_ns_c[c], (int)(so[i + 1] - so[i]));
        const bool fits = events_fast_smem_bytes(max_ns_c[c], max_nz, w, fast_max_d_for(w, max_nz)) <= kMaxSmemOptin;
        for (int i = 0; i < n_events; ++i) {
            if (fast_warps_for((int)(so[i + 1] - so[i])) != w) continue;
            if (fits && tk_h[i] > 0.0 && udz[i] > 0.0) { fast_ev.push_back(i); ++n_fast_c[c]; }
            else slow_ev.push_back(i);
        }
    }
    std::sort(slow_ev.begin(), slow_ev.end());
    // replace the previous set
    cudaStreamSynchronize(ctx->stream);
    free_pool(ctx->owned_grp);
    ctx->n_groups = 0;
    ctx->grp_off = nullptr; ctx->grp_lnf = nullptr;
    free_pool(ctx->owned_ev);
    drop_work(ctx);
    ctx->have_events = false;
    EventSetDev E{};
    E.n_events = n_events; E.max_ns = max_ns; E.max_nz = max_nz;
    CK(upload(ctx->owned_ev, &E.sample_off, so)); CK(upload(ctx->owned_ev, &E.grid_off, go));
    CK(upload(ctx->owned_ev, &E.rec, rec));
    CK(upload(ctx->owned_ev, &E.k_lo, k_lo)); CK(upload(ctx->owned_ev, &E.k_hi, k_hi));
    CK(upload(ctx->owned_ev, &E.perm, perm)); CK(upload(ctx->owned_ev, &E.zc, zc)); CK(upload(ctx->owned_ev, &E.qn, qn));
    CK(upload(ctx->owned_ev, &E.uni_dz, udz)); CK(upload(ctx->owned_ev, &E.max_dz, maxdz));
    CK(upload(ctx->owned_ev, &E.ep_q0, ep0)); CK(upload(ctx->owned_ev, &E.ep_q1, ep1)); CK(upload(ctx->owned_ev, &E.ep_q2, ep2));
    CK(upload(ctx->owned_ev, &E.lnm1_lo, lm_lo)); CK(upload(ctx->owned_ev, &E.lnm1_hi, lm_hi)); CK(upload(ctx->owned_ev, &E.chunk_top, chunk_top));
    CK(upload(ctx->owned_ev, &E.z0, z0));
    CK(upload(ctx->owned_ev, &E.tk_c, tk_c)); CK(upload(ctx->owned_ev, &E.tk_h, tk_h));
    CK(upload(ctx->owned_ev, &E.poly_off, poff)); CK(upload(ctx->owned_ev, &E.prec_a, prec_a)); CK(upload(ctx->owned_ev, &E.prec_b, prec_b));
    if (fixed_bw) CK(upload(ctx->owned_ev, &E.fixed_bw, h_bw));
    CK(upload(ctx->owned_ev, &E.qn4, qn4)); CK(upload(ctx->owned_ev, &E.q4_off, q4off));
    CK(upload(ctx->owned_ev, &ctx->fast_ev, fast_ev)); CK(upload(ctx->owned_ev, &ctx->slow_ev, slow_ev));
    ctx->n_fast = (int)fast_ev.size(); ctx->n_slow = (int)slow_ev.size();
    for (int c = 0; c < kFastClasses; ++c) { ctx->n_fast_c[c] = n_fast_c[c]; ctx->max_ns_c[c] = max_ns_c[c]; }
    CK(upload(ctx->owned_ev, &ctx->ev_ln_shift, shift));
    CK(upload(ctx->owned_ev, &ctx->ev_ln_qscale, qshift));
    ctx->ev = E;
    ctx->ev_m_top = m_top;
    ctx->ev_grid = grid;
    ctx->h_sample_off = so;
    ctx->h_grid_off = go;
    ctx->have_events = true;
    return CHIM_OK;
}

int chim_set_event_groups(chim_ctx* ctx, int32_t n_groups, const int64_t* group_off, const double* ln_factor) {
    if (!ctx) return CHIM_EINVAL;
    if (!ctx->have_events) return fail(ctx, CHIM_ESTATE, "chim_set_event_groups: call chim_init_events first");
    CK(cudaSetDevice(ctx->cfg.device));
    if (n_groups < 0 || (n_groups > 0 && (!group_off || !ln_factor)))
        return fail(ctx, CHIM_EINVAL, "chim_set_event_groups: null pointer or n_groups < 0");
    std::vector<int64_t> go;
    std::vector<double> lf;
    if (n_groups > 0) {
        CK(fetch(ctx, group_off, (size_t)n_groups + 1, go));
        CK(fetch(ctx, ln_factor, (size_t)ctx->ev.n_events, lf));
        if (go[0] != 0 || go[n_groups] != ctx->ev.n_events)
            return fail(ctx, CHIM_EINVAL, "chim_set_event_groups: group_off must start at 0 and end at n_events");
        for (int g = 0; g < n_groups; ++g)
            if (!(go[g + 1] > go[g])) return fail(ctx, CHIM_EINVAL, "chim_set_event_groups: group_off must be strictly increasing");
        if (!all_finite(lf)) return fail(ctx, CHIM_EINVAL, "chim_set_event_groups: non-finite ln_factor");
    }
    cudaStreamSynchronize(ctx->stream);
    free_pool(ctx->owned_grp);
    ctx->n_groups = 0;
    ctx->grp_off = nullptr; ctx->grp_lnf = nullptr;
    if (n_groups > 0) {
        CK(upload(ctx->owned_grp, &ctx->grp_off, go));
        CK(upload(ctx->owned_grp, &ctx->grp_lnf, lf));
        ctx->n_groups = n_groups;
    }
    return CHIM_OK;
}

// eq. 8 (and, with a completeness map, eq. 7, 9, 10) on redshift grids; shared by chim_build_pcat / chim_build_pgal
static int build_pgal_impl(chim_ctx* ctx, const char* who, double omega_m, double z_max, int32_t n_los, const int64_t* gal_off,
                           const double* z_gal, const double* sigma_gal, const double* w_gal, const int64_t* compl_off,
                           const double* z_compl, const double* p_compl, const int64_t* grid_off, const double* z_grid,
                           double* p_out, double* f_r_out) {
    const std::string W(who);
    if (!ctx) return CHIM_EINVAL;
    if (n_los < 1 || !gal_off || !z_gal || !sigma_gal || !grid_off || !z_grid || !p_out || !(omega_m > 0.0) || !(omega_m <= 1.0))
        return fail(ctx, CHIM_EINVAL, W + ": null pointer, n_los < 1 or omega_m outside (0, 1]");
    const bool with_compl = compl_off != nullptr;
    if (with_compl && (!z_compl || !p_compl || !(z_max > 0.0) || !std::isfinite(z_max)))
        return fail(ctx, CHIM_EINVAL, W + ": null completeness arrays or z_max <= 0");
    CK(cudaSetDevice(ctx->cfg.device));
    std::vector<int64_t> go, po, co;
    CK(fetch(ctx, gal_off, (size_t)n_los + 1, go));
    CK(fetch(ctx, grid_off, (size_t)n_los + 1, po));
    if (with_compl) CK(fetch(ctx, compl_off, (size_t)n_los + 1, co));
    if (go[0] != 0 || po[0] != 0 || (with_compl && co[0] != 0)) return fail(ctx, CHIM_EINVAL, W + ": offsets must start at 0");
    for (int i = 0; i < n_los; ++i) {
        if (go[i + 1] <= go[i] || po[i + 1] < po[i])
            return fail(ctx, CHIM_EINVAL, W + ": every line of sight needs >= 1 galaxy; offsets must not decrease");
        if (with_compl && co[i + 1] - co[i] < 2) return fail(ctx, CHIM_EINVAL, W + ": every line of sight needs >= 2 completeness nodes");
    }
    const size_t NG = (size_t)go[n_los], NP = (size_t)po[n_los], NC = with_compl ? (size_t)co[n_los] : 0;
    std::vector<double> hz, hs, hw, hg, hzc, hpc;
    CK(fetch(ctx, z_gal, NG, hz)); CK(fetch(ctx, sigma_gal, NG, hs)); CK(fetch(ctx, z_grid, NP, hg));
    if (w_gal) CK(fetch(ctx, w_gal, NG, hw));
    if (with_compl) { CK(fetch(ctx, z_compl, NC, hzc)); CK(fetch(ctx, p_compl, NC, hpc)); }
    if (!all_finite(hz) || !all_finite(hs) || !all_finite(hw) || !all_finite(hg) || !all_finite(hzc) || !all_finite(hpc))
        return fail(ctx, CHIM_EINVAL, W + ": non-finite input");
    for (size_t g = 0; g < NG; ++g)
        if (hz[g] < 0.0 || !(hs[g] > 0.0) || (w_gal && !(hw[g] > 0.0)))
            return fail(ctx, CHIM_EINVAL, W + ": need z_gal >= 0, sigma_gal > 0, w_gal > 0");
    for (size_t i = 0; i < NP; ++i)
        if (hg[i] < 0.0) return fail(ctx, CHIM_EINVAL, W + ": z_grid must be >= 0");
    if (with_compl)
        for (int i = 0; i < n_los; ++i)
            for (int64_t k = co[i]; k < co[i + 1]; ++k)
                if (hpc[k] < 0.0 || hpc[k] > 1.0 || hzc[k] < 0.0 || (k > co[i] && !(hzc[k] > hzc[k - 1])))
                    return fail(ctx, CHIM_EINVAL, W + ": need 0 <= P_compl <= 1 on strictly increasing z_compl >= 0");
    std::vector<void*> pool;
    const int64_t *d_go = nullptr, *d_po = nullptr, *d_co = nullptr;
    const double *d_z = nullptr, *d_s = nullptr, *d_w = nullptr, *d_g = nullptr, *d_zc = nullptr, *d_pc = nullptr;
    double *d_coef = nullptr, *d_out = nullptr, *d_fr = nullptr;
    cudaError_t e = upload(pool, &d_go, go);
    if (e == cudaSuccess) e = upload(pool, &d_po, po);
    if (e == cudaSuccess) e = upload(pool, &d_z, hz);
    if (e == cudaSuccess) e = upload(pool, &d_s, hs);
    if (e == cudaSuccess && w_gal) e = upload(pool, &d_w, hw);
    if (e == cudaSuccess) e = upload(pool, &d_g, hg);
    if (e == cudaSuccess) e = dev_alloc(pool, &d_coef, NG);
    if (e == cudaSuccess) e = dev_alloc(pool, &d_out, NP);
    if (e == cudaSuccess && with_compl) e = upload(pool, &d_co, co);
    if (e == cudaSuccess && with_compl) e = upload(pool, &d_zc, hzc);
    if (e == cudaSuccess && with_compl) e = upload(pool, &d_pc, hpc);
    if (e == cudaSuccess && with_compl) e = dev_alloc(pool, &d_fr, (size_t)n_los);
    if (e == cudaSuccess) e = launch_pcat(omega_m, n_los, d_go, d_z, d_s, d_w, d_po, d_g, d_coef, d_out, ctx->stream);
    if (e == cudaSuccess && with_compl) e = launch_pgal(omega_m, z_max, n_los, d_co, d_zc, d_pc, d_po, d_g, d_out, d_fr, ctx->stream);
    if (e == cudaSuccess) e = cudaStreamSynchronize(ctx->stream);
    const cudaMemcpyKind back = ctx->cfg.mem == CHIM_MEM_DEVICE ? cudaMemcpyDeviceToDevice : cudaMemcpyDeviceToHost;
    if (e == cudaSuccess && NP > 0) e = cudaMemcpy(p_out, d_out, NP * sizeof(double), back);
    if (e == cudaSuccess && with_compl && f_r_out) e = cudaMemcpy(f_r_out, d_fr, (size_t)n_los * sizeof(double), back);
    free_pool(pool);
    if (e != cudaSuccess) return cuda_fail(ctx, e, who);
    return CHIM_OK;
}

int chim_build_pcat(chim_ctx* ctx, double omega_m, int32_t n_los, const int64_t* gal_off, const double* z_gal,
                    const double* sigma_gal, const double* w_gal, const int64_t* grid_off, const double* z_grid,
                    double* p_cat_out) {
    return build_pgal_impl(ctx, "chim_build_pcat", omega_m, 0.0, n_los, gal_off, z_gal, sigma_gal, w_gal, nullptr, nullptr, nullptr,
                           grid_off, z_grid, p_cat_out, nullptr);
}

int chim_build_pgal(chim_ctx* ctx, double omega_m, double z_max, int32_t n_los, const int64_t* gal_off, const double* z_gal,
                    const double* sigma_gal, const double* w_gal, const int64_t* compl_off, const double* z_compl,
                    const double* p_compl, const int64_t* grid_off, const double* z_grid, double* p_gal_out, double* f_r_out) {
    if (ctx && !compl_off) return fail(ctx, CHIM_EINVAL, "chim_build_pgal: compl_off is NULL (use chim_build_pcat for a complete catalogue)");
    return build_pgal_impl(ctx, "chim_build_pgal", omega_m, z_max, n_los, gal_off, z_gal, sigma_gal, w_gal, compl_off, z_compl, p_compl,
                           grid_off, z_grid, p_gal_out, f_r_out);
}

// eq. 8 for callers that cannot allocate (include/chim.h; k_pcat_static.cu): device pointers only, enqueue-only, and on this
// path no cudaMalloc / cudaFree / host copy -- the failure messages below are the only place that touches the host heap.
int chim_build_pcat_static(chim_ctx* ctx, double omega_m, int32_t n_los, int64_t n_gal_total, const int64_t* gal_off,
                           const double* z_gal, const double* sigma_gal, const double* w_gal, const int64_t* grid_off,
                           const double* z_grid, double* p_cat_out) {
    if (!ctx) return CHIM_EINVAL;
    if (n_los < 1 || !gal_off || !z_gal || !sigma_gal || !grid_off || !z_grid || !p_cat_out || !(omega_m > 0.0) || !(omega_m <= 1.0))
        return fail(ctx, CHIM_EINVAL, "chim_build_pcat_static: null pointer, n_los < 1 or omega_m outside (0, 1]");
    if (n_gal_total < n_los)
        return fail(ctx, CHIM_EINVAL, "chim_build_pcat_static: n_gal_total < n_los (every line of sight needs >= 1 galaxy)");
    if (n_gal_total > (int64_t)pcat_static_max_galaxies())
        return fail(ctx, CHIM_EINVAL, "chim_build_pcat_static: n_gal_total = " + std::to_string(n_gal_total) +
                                          " exceeds CHIM_PCAT_STATIC_MAX_GALAXIES = " + std::to_string(pcat_static_max_galaxies()) +
                                          " (the fixed scratch array); split the lines of sight over several calls or use chim_build_pcat");
    CK(cudaSetDevice(ctx->cfg.device));
    cudaError_t e = launch_pcat_static(omega_m, n_los, (long long)n_gal_total, gal_off, z_gal, sigma_gal, w_gal, grid_off, z_grid,
                                       p_cat_out, ctx->stream);
    if (e != cudaSuccess) return cuda_fail(ctx, e, "chim_build_pcat_static");
    return CHIM_OK;
}

int chim_init_injections(chim_ctx* ctx, int64_t n_det, int64_t n_inj_total, const double* dL, const double* m1d,
                         const double* m2d, const double* ln_pdraw) {
    if (!ctx) return CHIM_EINVAL;
    CK(cudaSetDevice(ctx->cfg.device));
    if (n_det == 0) {
        cudaStreamSynchronize(ctx->stream);
        free_pool(ctx->owned_inj);
        drop_work(ctx);
        ctx->have_inj = false;
        ctx->inj_blocks = 0;
        return CHIM_OK;
    }
    if (n_det < 0 || n_inj_total < n_det || !dL || !m1d || !m2d || !ln_pdraw)
        return fail(ctx, CHIM_EINVAL, "chim_init_injections: null pointer, n_det < 0 or n_inj_total < n_det");
    const size_t N = (size_t)n_det;
    std::vector<double> h_dl, h_m1, h_m2, h_lp;
    CK(fetch(ctx, dL, N, h_dl)); CK(fetch(ctx, m1d, N, h_m1)); CK(fetch(ctx, m2d, N, h_m2)); CK(fetch(ctx, ln_pdraw, N, h_lp));
    if (!all_finite(h_dl) || !all_finite(h_m1) || !all_finite(h_m2) || !all_finite(h_lp))
        return fail(ctx, CHIM_EINVAL, "chim_init_injections: non-finite input");
    double xmin = INFINITY, xmax = -INFINITY, sh = -INFINITY, m_top = 0.0;
    for (size_t j = 0; j < N; ++j) {
        if (!(h_dl[j] > 0.0) || !(h_m2[j] > 0.0) || !(h_m1[j] >= h_m2[j]))
            return fail(ctx, CHIM_EINVAL, "chim_init_injections: need dL > 0 and m1d >= m2d > 0");
        m_top = std::max(m_top, h_m1[j]);
        double x = std::log(h_dl[j]);
        xmin = std::min(xmin, x);
        xmax = std::max(xmax, x);
        sh = std::max(sh, -h_lp[j]);
    }
    DlGrid grid = make_dl_grid(xmin, xmax, choose_dl_intervals(ctx, xmin, xmax));
    const double l2e = 1.4426950408889634074;
    std::vector<int64_t> idx(N);
    std::iota(idx.begin(), idx.end(), (int64_t)0);
    std::stable_sort(idx.begin(), idx.end(), [&](int64_t a, int64_t b) { return h_dl[a] < h_dl[b]; });
    std::vector<float4> rec(2 * N);
    for (size_t j = 0; j < N; ++j) {
        const size_t o = (size_t)idx[j];
        const double tk = (std::log(h_dl[o]) - grid.x0) / grid.dx + 1.0;
        const int k = std::min(std::max((int)tk, 1), grid.K);
        rec[2 * j] = make_float4(bits_f((uint32_t)k), (float)(tk - (double)k), (float)h_m1[o], (float)h_m2[o]);
        rec[2 * j + 1] = make_float4((float)std::log(h_m1[o]), (float)std::log(h_m2[o] / h_m1[o]), (float)(l2e * (-h_lp[o] - sh)), 0.f);
    }
    // chunk-local polynomials of k_inject: the set is sorted in d_L, so a chunk of kInjChunk injections spans a narrow range
    const int n_chunks = (int)((n_det + kInjChunk - 1) / kInjChunk);
    std::vector<float4> prec_a((size_t)n_chunks * kInjChunk + 2048, make_float4(1.f, 1.f, 0.f, 0.f));   // + spare tail (prefetch)
    std::vector<float2> prec_b((size_t)n_chunks * kInjChunk + 2048, make_float2(0.f, 0.f));
    std::vector<double> ctk_c(n_chunks), ctk_h(n_chunks);
    std::vector<float> blk_m2d((size_t)n_chunks * (kInjChunk / 256), INFINITY);
    for (int c = 0; c < n_chunks; ++c) {
        const size_t a = (size_t)c * kInjChunk, b = std::min<size_t>(a + kInjChunk, N);
        auto tk_of = [&](size_t j) { return (double)f_bits(rec[2 * j].x) + (double)rec[2 * j].y; };   // k + t
        const double lo = tk_of(a), hi = tk_of(b - 1);                // (still in d_L order here)
        {   // inside the chunk the order is free: by m2d, so that the warps of k_inject are uniform in "m2 below m_low" and
            // "m2 inside the smoothing window" (1 + z varies by a few percent over a chunk)
            std::vector<size_t> ord(b - a);
            std::iota(ord.begin(), ord.end(), a);
            std::stable_sort(ord.begin(), ord.end(), [&](size_t x, size_t y) { return h_m2[(size_t)idx[x]] < h_m2[(size_t)idx[y]]; });
            // ... and inside every block of 256 by m1d: the 32 lanes of a warp then address neighbouring rows of the mass table
            // (shared-memory bank conflicts of the 16-byte row loads: 9 -> ~4 wavefronts)
            for (size_t q = 0; q < ord.size(); q += 256)
                std::stable_sort(ord.begin() + q, ord.begin() + std::min(q + 256, ord.size()),
                                 [&](size_t x, size_t y) { return h_m1[(size_t)idx[x]] < h_m1[(size_t)idx[y]]; });
            std::vector<float4> r2(2 * (b - a));
            std::vector<int64_t> i2(b - a);
            for (size_t k = 0; k < b - a; ++k) { r2[2 * k] = rec[2 * ord[k]]; r2[2 * k + 1] = rec[2 * ord[k] + 1]; i2[k] = idx[ord[k]]; }
            std::copy(r2.begin(), r2.end(), rec.begin() + 2 * a);
            std::copy(i2.begin(), i2.end(), idx.begin() + a);
        }
        const double half = 0.5 * (hi - lo) * (1.0 + 1e-9) + 1e-3;
        ctk_c[c] = 0.5 * (lo + hi);
        ctk_h[c] = (half * grid.dx <= kPolyMaxHalfRange) ? half : 0.0;
        for (int k = 0; k < kInjChunk / 256; ++k) {   // largest m2d of every block of 256 (rounded up: the test in k_inject is conservative)
            const size_t e = std::min<size_t>(a + (size_t)(k + 1) * 256, b);
            float mxb = 0.f;
            for (size_t q = a + (size_t)k * 256; q < e; ++q) mxb = std::max(mxb, (float)h_m2[(size_t)idx[q]]);
            blk_m2d[(size_t)c * (kInjChunk / 256) + k] = (e > a + (size_t)k * 256) ? std::nextafter(mxb, INFINITY) : INFINITY;
        }
        for (size_t j = a; j < a + kInjChunk; ++j) {
            const size_t js = std::min(j, b - 1), o = (size_t)idx[js];
            const double t = (tk_of(js) - ctk_c[c]) / half;
            prec_a[j] = make_float4((float)h_m1[o], (float)h_m2[o], (float)t, (float)std::log(h_m1[o]));
            prec_b[j] = make_float2((float)std::log(h_m2[o]), rec[2 * js + 1].z);
        }
    }
    cudaStreamSynchronize(ctx->stream);
    free_pool(ctx->owned_inj);
    drop_work(ctx);
    ctx->have_inj = false;
    InjSetDev I{};
    I.n_det = n_det;
    I.n_inj_total = (double)n_inj_total;
    CK(upload(ctx->owned_inj, &I.rec, rec));
    CK(upload(ctx->owned_inj, &I.perm, idx));
    CK(upload(ctx->owned_inj, &I.prec_a, prec_a)); CK(upload(ctx->owned_inj, &I.prec_b, prec_b));
    CK(upload(ctx->owned_inj, &I.tk_c, ctk_c)); CK(upload(ctx->owned_inj, &I.tk_h, ctk_h));
    CK(upload(ctx->owned_inj, &I.blk_m2d, blk_m2d));
    ctx->inj = I;
    ctx->inj_m_top = m_top;
    ctx->inj_grid = grid;
    ctx->inj_ln_shift = sh;
    ctx->inj_blocks = (int)((n_det + kInjChunk - 1) / kInjChunk);
    ctx->have_inj = true;
    return CHIM_OK;
}

int chim_loglike_batch(chim_ctx* ctx, int32_t n_lambda, const double* lambda, double* out_loglike, double* out_event_logI,
                       double* out_logxi, double* out_neff, uint32_t* out_flags) {
    if (!ctx) return CHIM_EINVAL;
    if (!ctx->have_events) return fail(ctx, CHIM_ESTATE, "chim_loglike_batch: call chim_init_events first");
    if (n_lambda < 0 || (n_lambda > 0 && (!lambda || !out_loglike)))
        return fail(ctx, CHIM_EINVAL, "chim_loglike_batch: null lambda/out_loglike or n_lambda < 0");
    if (n_lambda == 0) return CHIM_OK;
    CK(cudaSetDevice(ctx->cfg.device));
    // (a work-list entry holds lambda x n_events + event in 31 bits)
    const int chunk = (int)std::min<long long>(std::min<int>(ctx->cfg.lambda_chunk, n_lambda), std::max<long long>(1, 0x7FFFFFFFLL / std::max(ctx->ev.n_events, 1)));
    int rc = ensure_work(ctx, chunk);
    if (rc != CHIM_OK) return rc;
    ctx->launches = 0;
    ctx->ev_kind.clear();
    CK(cudaMemsetAsync(ctx->stats, 0, 4 * sizeof(unsigned long long), ctx->stream));
    const int n_chunks = (n_lambda + chunk - 1) / chunk;
    // several chunks: S1 of chunk c + 1 on the auxiliary stream while S2-S6 of chunk c run (with per-kernel timing on, everything
    // stays on the context's stream, one kernel after the other, so that the times add up)
    const bool overlap = n_chunks > 1 && !ctx->profiling && ctx->aux_stream != nullptr;
    auto lam_of = [&](int c) { return lambda + (size_t)c * chunk * CHIM_N_LAMBDA_PARAMS; };
    auto nl_of = [&](int c) { return std::min(chunk, n_lambda - c * chunk); };
    if (overlap) {
        CK(cudaEventRecord(ctx->ev_begin, ctx->stream));
        CK(cudaStreamWaitEvent(ctx->aux_stream, ctx->ev_begin, 0));
        use_s1_set(ctx, 0);
        rc = run_s1(ctx, nl_of(0), lam_of(0), ctx->aux_stream);
        if (rc != CHIM_OK) return rc;
        CK(cudaEventRecord(ctx->ev_s1[0], ctx->aux_stream));
    }
    for (int c = 0; c < n_chunks; ++c) {
        const int c0 = c * chunk, nl = nl_of(c), k = c & 1;
        if (overlap) {
            CK(cudaStreamWaitEvent(ctx->stream, ctx->ev_s1[k], 0));
            if (c + 1 < n_chunks) {
                if (c >= 1) CK(cudaStreamWaitEvent(ctx->aux_stream, ctx->ev_rest[k ^ 1], 0));   // (chunk c - 1 has left that set)
                use_s1_set(ctx, k ^ 1);
                rc = run_s1(ctx, nl_of(c + 1), lam_of(c + 1), ctx->aux_stream);
                if (rc != CHIM_OK) return rc;
                CK(cudaEventRecord(ctx->ev_s1[k ^ 1], ctx->aux_stream));
            }
            use_s1_set(ctx, k);
        } else {
            use_s1_set(ctx, 0);
            rc = run_s1(ctx, nl, lam_of(c), ctx->stream);
            if (rc != CHIM_OK) return rc;
        }
        rc = run_rest(ctx, nl, out_loglike + c0, out_event_logI ? out_event_logI + (size_t)c0 * ctx->ev.n_events : nullptr,
                      out_logxi ? out_logxi + c0 : nullptr, out_neff ? out_neff + c0 : nullptr, out_flags ? out_flags + c0 : nullptr);
        if (rc != CHIM_OK) return rc;
        if (overlap) CK(cudaEventRecord(ctx->ev_rest[k], ctx->stream));
    }
    use_s1_set(ctx, 0);
    ctx->last.kde_pairs_dense = 0;
    for (int i = 0; i < ctx->ev.n_events; ++i)
        ctx->last.kde_pairs_dense += (uint64_t)(ctx->h_sample_off[i + 1] - ctx->h_sample_off[i]) *
                                     (uint64_t)(ctx->h_grid_off[i + 1] - ctx->h_grid_off[i]);
    ctx->last.kde_pairs_dense *= (uint64_t)n_lambda;
    ctx->last.sample_evals = (uint64_t)ctx->h_sample_off[ctx->ev.n_events] * (uint64_t)n_lambda;
    ctx->last.injection_evals = ctx->have_inj ? (uint64_t)ctx->inj.n_det * (uint64_t)n_lambda : 0;
    ctx->last.kernel_launches = ctx->launches;
    return CHIM_OK;
}

int chim_loglike_batch_host(chim_ctx* ctx, int32_t n_lambda, const double* lambda, double* out_loglike,
                            double* out_event_logI, double* out_logxi, double* out_neff, uint32_t* out_flags) {
    if (!ctx) return CHIM_EINVAL;
    if (!ctx->have_events) return fail(ctx, CHIM_ESTATE, "chim_loglike_batch_host: call chim_init_events first");
    if (n_lambda < 0 || (n_lambda > 0 && (!lambda || !out_loglike)))
        return fail(ctx, CHIM_EINVAL, "chim_loglike_batch_host: null lambda/out_loglike or n_lambda < 0");
    if (n_lambda == 0) return CHIM_OK;
    CK(cudaSetDevice(ctx->cfg.device));
    if (n_lambda > ctx->host_nl) {
        cudaStreamSynchronize(ctx->stream);
        free_pool(ctx->owned_host);
        ctx->host_nl = 0;
        CK(dev_alloc(ctx->owned_host, &ctx->st_lam, (size_t)n_lambda * CHIM_N_LAMBDA_PARAMS));
        CK(dev_alloc(ctx->owned_host, &ctx->st_ll, n_lambda));
        CK(dev_alloc(ctx->owned_host, &ctx->st_ev, (size_t)n_lambda * ctx->ev.n_events));
        CK(dev_alloc(ctx->owned_host, &ctx->st_xi, n_lambda));
        CK(dev_alloc(ctx->owned_host, &ctx->st_neff, n_lambda));
        CK(dev_alloc(ctx->owned_host, &ctx->st_fl, n_lambda));
        ctx->host_nl = n_lambda;
    }
    cudaStream_t st = ctx->stream;
    CK(cudaMemcpyAsync(ctx->st_lam, lambda, sizeof(double) * n_lambda * CHIM_N_LAMBDA_PARAMS, cudaMemcpyHostToDevice, st));
    int rc = chim_loglike_batch(ctx, n_lambda, ctx->st_lam, ctx->st_ll, out_event_logI ? ctx->st_ev : nullptr,
                                out_logxi ? ctx->st_xi : nullptr, out_neff ? ctx->st_neff : nullptr,
                                out_flags ? ctx->st_fl : nullptr);
    if (rc != CHIM_OK) return rc;
    CK(cudaMemcpyAsync(out_loglike, ctx->st_ll, sizeof(double) * n_lambda, cudaMemcpyDeviceToHost, st));
    if (out_event_logI)
        CK(cudaMemcpyAsync(out_event_logI, ctx->st_ev, sizeof(double) * n_lambda * ctx->ev.n_events, cudaMemcpyDeviceToHost, st));
    if (out_logxi) CK(cudaMemcpyAsync(out_logxi, ctx->st_xi, sizeof(double) * n_lambda, cudaMemcpyDeviceToHost, st));
    if (out_neff) CK(cudaMemcpyAsync(out_neff, ctx->st_neff, sizeof(double) * n_lambda, cudaMemcpyDeviceToHost, st));
    if (out_flags) CK(cudaMemcpyAsync(out_flags, ctx->st_fl, sizeof(uint32_t) * n_lambda, cudaMemcpyDeviceToHost, st));
    CK(cudaStreamSynchronize(st));
    return CHIM_OK;
}

int chim_loglike_grad_batch(chim_ctx* ctx, int32_t n_lambda, const double* lambda, double rel_step, double* out_loglike,
                            double* out_grad, uint32_t* out_flags) {
    if (!ctx) return CHIM_EINVAL;
    if (!ctx->have_events) return fail(ctx, CHIM_ESTATE, "chim_loglike_grad_batch: call chim_init_events first");
    if (n_lambda < 0 || (n_lambda > 0 && (!lambda || !out_loglike || !out_grad)))
        return fail(ctx, CHIM_EINVAL, "chim_loglike_grad_batch: null lambda / out_loglike / out_grad or n_lambda < 0");
    if (!(rel_step > 0.0) || !(rel_step < 0.5)) return fail(ctx, CHIM_EINVAL, "chim_loglike_grad_batch: rel_step must be in (0, 0.5)");
    if (n_lambda == 0) return CHIM_OK;
    const int R = grad_rows();
    if ((long long)n_lambda * R > (1LL << 30)) return fail(ctx, CHIM_EINVAL, "chim_loglike_grad_batch: n_lambda too large");
    CK(cudaSetDevice(ctx->cfg.device));
    if (n_lambda > ctx->grad_nl) {
        cudaStreamSynchronize(ctx->stream);
        free_pool(ctx->owned_grad);
        ctx->grad_nl = 0;
        CK(dev_alloc(ctx->owned_grad, &ctx->g_lam, (size_t)n_lambda * R * CHIM_N_LAMBDA_PARAMS));
        CK(dev_alloc(ctx->owned_grad, &ctx->g_ll, (size_t)n_lambda * R));
        CK(dev_alloc(ctx->owned_grad, &ctx->g_fl, (size_t)n_lambda * R));
        ctx->grad_nl = n_lambda;
    }
    CK(launch_grad_expand(lambda, n_lambda, rel_step, ctx->g_lam, ctx->stream));
    int rc = chim_loglike_batch(ctx, n_lambda * R, ctx->g_lam, ctx->g_ll, nullptr, nullptr, nullptr, ctx->g_fl);
    if (rc != CHIM_OK) return rc;
    CK(launch_grad_combine(lambda, n_lambda, rel_step, ctx->g_ll, ctx->g_fl, out_loglike, out_grad, out_flags, ctx->stream));
    ctx->last.kernel_launches += 2;
    return CHIM_OK;
}

int chim_get_stats(chim_ctx* ctx, chim_stats* out) {
    if (!ctx || !out) return CHIM_EINVAL;
    if (!ctx->stats) return fail(ctx, CHIM_ESTATE, "chim_get_stats: no batch has run");
    CK(cudaSetDevice(ctx->cfg.device));
    CK(cudaStreamSynchronize(ctx->stream));
    unsigned long long s[4];
    CK(cudaMemcpy(s, ctx->stats, sizeof s, cudaMemcpyDeviceToHost));
    ctx->last.kde_pairs_evaluated = s[0];
    ctx->last.kde_pairs_in_cutoff = s[1];
    *out = ctx->last;
    return CHIM_OK;
}

int chim_set_profiling(chim_ctx* ctx, int32_t enable) {
    if (!ctx) return CHIM_EINVAL;
    ctx->profiling = enable != 0;
    ctx->ev_kind.clear();
    return CHIM_OK;
}

int chim_get_kernel_times(chim_ctx* ctx, chim_kernel_times* out) {
    if (!ctx || !out) return CHIM_EINVAL;
    CK(cudaSetDevice(ctx->cfg.device));
    CK(cudaStreamSynchronize(ctx->stream));
    std::memset(out, 0, sizeof(*out));
    double* ms[5] = {&out->tables_ms, &out->events_ms, &out->inject_ms, &out->combine_ms, &out->events_general_ms};
    uint32_t* nl[5] = {&out->tables_launches, &out->events_launches, &out->inject_launches, &out->combine_launches, &out->events_general_launches};
    for (size_t i = 0; i < ctx->ev_kind.size(); ++i) {
        float t = 0.f;
        CK(cudaEventElapsedTime(&t, ctx->ev_pool[2 * i], ctx->ev_pool[2 * i + 1]));
        *ms[ctx->ev_kind[i]] += t;
        *nl[ctx->ev_kind[i]] += 1;
    }
    if (ctx->work_count) {
        unsigned int n = 0;
        CK(cudaMemcpy(&n, ctx->work_count, sizeof n, cudaMemcpyDeviceToHost));
        out->events_handed_over = n;
    }
    return CHIM_OK;
}

int chim_measure_alu_peaks(chim_ctx* ctx, chim_alu_peaks* out) {
    if (!ctx || !out) return CHIM_EINVAL;
    CK(cudaSetDevice(ctx->cfg.device));
    cudaDeviceProp prop;
    CK(cudaGetDeviceProperties(&prop, ctx->cfg.device));
    double g[4];
    CK(measure_alu_peaks(prop.multiProcessorCount, 3, ctx->stream, g));
    out->ex2_gops = g[0]; out->ffma_gops = g[1]; out->dfma_gops = g[2]; out->ffma2_gops = g[3];
    out->sm_count = prop.multiProcessorCount;
    out->reserved = 0;
    return CHIM_OK;
}

// ---- diagnostics --------------------------------------------------------------------------------------
static int debug_prepare(chim_ctx* ctx, const double* lambda, const char* who) {
    if (!ctx) return CHIM_EINVAL;
    if (!ctx->have_events) return fail(ctx, CHIM_ESTATE, std::string(who) + ": call chim_init_events first");
    if (!lambda) return fail(ctx, CHIM_EINVAL, std::string(who) + ": null lambda");
    CK(cudaSetDevice(ctx->cfg.device));
    int rc = ensure_work(ctx, 1);
    if (rc != CHIM_OK) return rc;
    TableParams TP = table_params(ctx);
    CK(cudaMemsetAsync(ctx->flags, 0, sizeof(uint32_t), ctx->stream));
    CK(launch_tables(lambda, 1, TP, ctx->Lc, ctx->dc_tab, ctx->tab_ev, ctx->tab_inj, ctx->mtab, ctx->stream));
    CK(launch_polyfit(ctx->Lc, ctx->tab_ev, ctx->ev_grid.rows(), 1, ctx->ev.n_events, ctx->ev.tk_c, ctx->ev.tk_h, ctx->ev.z0, 0.0, false,
                      ctx->poly_mats, ctx->ev.lnm1_lo, ctx->ev.lnm1_hi, ctx->cfg.n_mass_table,
                      events_mass_stage_rows(ctx->cfg.n_mass_table), ctx->ev_grid.dx, ctx->poly_ev, ctx->stream));
    if (ctx->have_inj)
        CK(launch_polyfit(ctx->Lc, ctx->tab_inj, ctx->inj_grid.rows(), 1, ctx->inj_blocks, ctx->inj.tk_c, ctx->inj.tk_h, nullptr,
                          ctx->cfg.z_cat_max, true, ctx->poly_mats, nullptr, nullptr, 0, 0, ctx->inj_grid.dx, ctx->poly_inj, ctx->stream));
    return CHIM_OK;
}

int chim_debug_table_lookup(chim_ctx* ctx, const double* lambda, int64_t n, const double* dL, double* z_out, double* ratio_out) {
    int rc = debug_prepare(ctx, lambda, "chim_debug_table_lookup");
    if (rc != CHIM_OK) return rc;
    if (n < 0 || (n > 0 && !dL)) return fail(ctx, CHIM_EINVAL, "chim_debug_table_lookup: bad arguments");
    CK(launch_table_lookup(ctx->Lc, ctx->tab_ev, ctx->ev_grid, n, dL, ctx->cfg.z_table_max, z_out, ratio_out, ctx->stream));
    CK(cudaStreamSynchronize(ctx->stream));
    return CHIM_OK;
}

static int debug_event(chim_ctx* ctx, const double* lambda, int32_t event, double* z_out, double* w_out, double* h_out,
                       double* K_out, double* logI_out, const char* who) {
    int rc = debug_prepare(ctx, lambda, who);
    if (rc != CHIM_OK) return rc;
    if (event < 0 || event >= ctx->ev.n_events) return fail(ctx, CHIM_EINVAL, std::string(who) + ": event out of range");
    if ((z_out == nullptr) != (w_out == nullptr)) return fail(ctx, CHIM_EINVAL, std::string(who) + ": z_out and w_out go together");
    EventKernelParams EP = event_params(ctx, 1);
    EP.dbg_event = event;
    EP.dbg_z = z_out; EP.dbg_w = w_out; EP.dbg_h = h_out; EP.dbg_K = K_out;
    if (K_out) CK(cudaMemsetAsync(K_out, 0, sizeof(double) * (size_t)(ctx->h_grid_off[event + 1] - ctx->h_grid_off[event]), ctx->stream));
    CK(launch_events(EP, true, ctx->stream));
    if (logI_out) CK(cudaMemcpyAsync(logI_out, ctx->logI, sizeof(double), cudaMemcpyDeviceToDevice, ctx->stream));
    CK(cudaStreamSynchronize(ctx->stream));
    return CHIM_OK;
}

int chim_debug_event_samples(chim_ctx* ctx, const double* lambda, int32_t event, double* z_out, double* w_out) {
    if (!z_out || !w_out) return fail(ctx, CHIM_EINVAL, "chim_debug_event_samples: null output");
    return debug_event(ctx, lambda, event, z_out, w_out, nullptr, nullptr, nullptr, "chim_debug_event_samples");
}

int chim_debug_event_kde(chim_ctx* ctx, const double* lambda, int32_t event, double* h_out, double* K_out, double* logI_out) {
    return debug_event(ctx, lambda, event, nullptr, nullptr, h_out, K_out, logI_out, "chim_debug_event_kde");
}

int chim_debug_injection_weights(chim_ctx* ctx, const double* lambda, double* s_out) {
    int rc = debug_prepare(ctx, lambda, "chim_debug_injection_weights");
    if (rc != CHIM_OK) return rc;
    if (!ctx->have_inj) return fail(ctx, CHIM_ESTATE, "chim_debug_injection_weights: no injections loaded");
    if (!s_out) return fail(ctx, CHIM_EINVAL, "chim_debug_injection_weights: null output");
    InjKernelParams IP{};
    IP.inj = ctx->inj; IP.Lc = ctx->Lc; IP.tab = ctx->tab_inj; IP.mtab = ctx->mtab;
    IP.n_lambda = 1; IP.tab_rows = ctx->inj_grid.rows(); IP.n_mass = ctx->cfg.n_mass_table; IP.chunk = kInjChunk;
    IP.z_table_max = ctx->cfg.z_table_max; IP.z_cat_max = ctx->cfg.z_cat_max;
    IP.partial = ctx->partial; IP.flags = ctx->flags; IP.dbg_s = s_out; IP.poly = ctx->poly_inj; IP.n_chunks = ctx->inj_blocks;
    IP.dbg_scale = std::exp(ctx->inj_ln_shift);
    CK(launch_inject(IP, ctx->inj_blocks, ctx->stream));
    CK(cudaStreamSynchronize(ctx->stream));
    return CHIM_OK;
}

}  // extern "C"
