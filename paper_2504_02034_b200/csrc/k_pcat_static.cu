// k_pcat_static.cu -- p_cat from galaxy lists (eq. 8; R22) without a single device allocation.
//
// Who this is for.  k_pcat (k_tables.cu) needs one double of scratch per galaxy (w_g / Z_g, the weight over the galaxy's own
// normalisation integral), and chim_build_pcat gets that scratch -- and device copies of everything else -- from cudaMalloc and
// gives it back with cudaFree.  Some users of this library must not do either while they run:
//   * a sampler living inside a JAX or PyTorch process whose framework has already reserved (nearly) all of the GPU's memory
//     for its own pool: a cudaMalloc from a foreign library then fails although the framework itself has plenty of room;
//   * a loop that rebuilds p_cat on the fly (another Omega_m, another catalogue cut) between likelihood batches and cannot
//     afford cudaMalloc / cudaFree there: both synchronise the whole device, so they stall the batch that is still running on the
//     context's streams (chim_loglike_batch itself is enqueue-only for that reason).
// For them the scratch of this variant is a fixed array in the library's own device image: it exists from the moment the
// library is loaded on a GPU until the process exits (kPcatStaticMax doubles = 2 MiB on every GPU that loads libchim.so,
// whether this entry point is ever called or not), and the caller passes device pointers for everything else.
//
// What follows from the array being shared:
//   * one array per GPU, shared by every context and every call.  Two calls that can overlap on the GPU (different streams,
//     different contexts, different host threads) race on it and both results are garbage.  Calls on one stream are safe.
//   * it keeps whatever the last call left in it.  Nothing in it has to start at zero: every line of sight writes the
//     coefficients of its own galaxies before it reads them (same CTA, one barrier in between), so it is never cleared.
//   * the first call on each GPU looks the array's device address up (cudaGetSymbolAddress, which may also load the kernel
//     image lazily).  Make that first call during start-up, before any stream capture and before the phase in which the
//     process must not touch the allocator; later calls only launch the kernel.
#include <mutex>

#include "chim_internal.cuh"

namespace chim {

namespace {

constexpr int kPcatStaticMax = CHIM_PCAT_STATIC_MAX_GALAXIES;
constexpr int kMaxDevices = 64;

// The scratch itself.  In host code this name is only a handle for the runtime's symbol calls -- it is NOT the device address
// (a kernel handed `g_pcat_coef` from the host faults, or quietly uses host memory where the GPU can reach it).  Host code
// gets the address from cudaGetSymbolAddress, once per device, below.
static __device__ __align__(256) double g_pcat_coef[kPcatStaticMax];

struct GLNodes { double x[kGLWin], w[kGLWin]; };   // Gauss-Legendre rule on [-1, 1], passed to the kernel by value (512 B)

// Nodes and weights of the n-point rule: roots of the Legendre polynomial P_n by Newton's iteration from the Chebyshev-like
// first guess, weights 2 / ((1 - x^2) P_n'(x)^2).
void legendre_pn(int n, double t, double* pn, double* dpn) {
    double pkm1 = 1.0, pk = t;
    for (int k = 1; k < n; ++k) {
        const double pkp1 = ((2 * k + 1) * t * pk - k * pkm1) / (k + 1);
        pkm1 = pk;
        pk = pkp1;
    }
    *pn = pk;
    *dpn = n * (pkm1 - t * pk) / (1.0 - t * t);
}
void fill_gauss_legendre(GLNodes* g) {
    const int n = kGLWin;
    const double pi = 3.14159265358979323846;
    for (int i = 0; i < (n + 1) / 2; ++i) {
        double t = cos(pi * (4 * i + 3) / (4.0 * n + 2.0)), pn, dpn;
        for (int it = 0; it < 64; ++it) {
            legendre_pn(n, t, &pn, &dpn);
            const double dt = pn / dpn;
            t -= dt;
            if (fabs(dt) < 1e-16) break;
        }
        legendre_pn(n, t, &pn, &dpn);
        g->x[i] = -t;
        g->x[n - 1 - i] = t;
        g->w[i] = g->w[n - 1 - i] = 2.0 / ((1.0 - t * t) * dpn * dpn);
    }
}

// V(z) = I(z)^2 / E(z), I = int_0^z dz'/E: dV_c/dz up to a constant that cancels in eq. 8 (as pcat_vol of k_tables.cu)
__device__ __forceinline__ double vol_static(double z, double Om, const GLNodes& gl) {
    double I = 0.0;
    const double hz = 0.5 * z;
#pragma unroll 4
    for (int q = 0; q < kGLWin; ++q) {
        const double a = 1.0 + hz * (1.0 + gl.x[q]);
        I += gl.w[q] * rsqrt(Om * a * a * a + 1.0 - Om);
    }
    I *= hz;
    const double a = 1.0 + z;
    return I * I * rsqrt(Om * a * a * a + 1.0 - Om);
}

// The variant of k_pcat: same arithmetic in the same order (one CTA per line of sight, fp64), with
//   coef = the address of g_pcat_coef as cudaGetSymbolAddress returned it on this device,
//   the quadrature rule in the kernel's parameters instead of the __constant__ tables chim_create fills, and
//   a check of the line of sight's galaxy range against the n_gal the host accepted, because nothing on the host has seen the
//   offsets: a range outside [0, n_gal] would leave the array, so that line of sight gets NaN on its whole grid instead.
__global__ void __launch_bounds__(256) k_pcat_static(double Om, GLNodes gl, long long n_gal, const int64_t* __restrict__ gal_off,
                                                     const double* __restrict__ zt, const double* __restrict__ st,
                                                     const double* __restrict__ wg, const int64_t* __restrict__ grid_off,
                                                     const double* __restrict__ zg, double* __restrict__ coef,
                                                     double* __restrict__ out) {
    __shared__ double red[256 / 32];
    __shared__ double s_sw;
    const int e = blockIdx.x, tid = threadIdx.x;
    const int64_t g0 = gal_off[e], g1 = gal_off[e + 1], p0 = grid_off[e], p1 = grid_off[e + 1];
    if (g0 < 0 || g1 <= g0 || g1 > n_gal) {                    // (CTA-uniform)
        for (int64_t i = p0 + tid; i < p1; i += 256) out[i] = NAN;
        return;
    }
    double sw = 0.0;
    for (int64_t g = g0 + tid; g < g1; g += 256) {
        const double m = zt[g], s = st[g], w = wg ? wg[g] : 1.0;
        const double lo = fmax(0.0, m - 10.0 * s), hi = m + 10.0 * s, hw = 0.5 * (hi - lo) / 8.0;
        double Z = 0.0;                                        // Z_g over [max(0, zt - 10 st), zt + 10 st], 8 panels of 32 nodes
        for (int p = 0; p < 8; ++p) {
            const double mid = lo + (2 * p + 1) * hw;
            double acc = 0.0;
            for (int q = 0; q < kGLWin; ++q) {
                const double z = mid + hw * gl.x[q], u = (z - m) / s;
                acc += gl.w[q] * exp(-0.5 * u * u) * vol_static(z, Om, gl);
            }
            Z += acc * hw;
        }
        coef[g] = w / Z;
        sw += w;
    }
    sw = warp_sum(sw);
    if ((tid & 31) == 0) red[tid >> 5] = sw;
    __syncthreads();                                           // also publishes this CTA's part of coef[]
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
            if (fabs(u) < 39.0) acc += coef[g] * exp(-0.5 * u * u);
        }
        out[i] = acc * inv_sw * vol_static(z, Om, gl);
    }
}

std::mutex g_setup_mu;
double* g_coef_addr[kMaxDevices] = {};     // device address of g_pcat_coef per CUDA ordinal (0 = not looked up yet)
GLNodes g_gl;
bool g_gl_ready = false;

}  // namespace

int pcat_static_max_galaxies() { return kPcatStaticMax; }

// Launches k_pcat_static on `st_` of the CURRENT device (the caller has made the right one current).  The first call on a
// device performs the one-off set-up described at the top of the file.  Returns cudaErrorInvalidValue for sizes the array
// cannot hold (the ABI entry point has already turned that into a readable message).  No cudaMalloc / cudaFree, no host heap.
cudaError_t launch_pcat_static(double Om, int n_los, long long n_gal, const int64_t* gal_off, const double* zt, const double* st,
                               const double* wg, const int64_t* grid_off, const double* zg, double* out, cudaStream_t st_) {
    if (n_los <= 0) return cudaSuccess;
    if (n_gal < 1 || n_gal > kPcatStaticMax) return cudaErrorInvalidValue;
    int dev = -1;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) return e;
    if (dev < 0 || dev >= kMaxDevices) return cudaErrorInvalidDevice;
    double* coef = nullptr;
    {
        std::lock_guard<std::mutex> lock(g_setup_mu);
        if (!g_gl_ready) { fill_gauss_legendre(&g_gl); g_gl_ready = true; }
        if (!g_coef_addr[dev]) {
            void* p = nullptr;
            e = cudaGetSymbolAddress(&p, g_pcat_coef);          // device `dev` is current: its copy of the array
            if (e != cudaSuccess) return e;
            if (!p) return cudaErrorInvalidSymbol;
            g_coef_addr[dev] = static_cast<double*>(p);
        }
        coef = g_coef_addr[dev];
    }
    k_pcat_static<<<n_los, 256, 0, st_>>>(Om, g_gl, n_gal, gal_off, zt, st, wg, grid_off, zg, coef, out);
    return cudaGetLastError();
}

}  // namespace chim
