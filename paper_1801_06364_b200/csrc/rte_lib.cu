// rte_lib.cu — C-ABI implementation (include/rte.h) of the B200-native P_N pseudospectral RTE stepper.
// Host logic + the non-hot kernels (layout transposes, coefficient maps, geometry generators, reductions);
// the hot per-axis pencil kernel lives in rte_pass.cuh, the register FFTs in rte_fft.cuh, the tables in rte_tables.h.
// No CPU fallback anywhere: every entry point that computes does so in a CUDA kernel or fails with RTE_ECUDA.
#include "../../include/rte.h"

#include <cuda_runtime.h>

#include <algorithm>
#include <cmath>
#include <cstddef>
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <limits>
#include <mutex>
#include <new>
#include <string>
#include <utility>
#include <vector>

#include "rte_pass.cuh"
#include "rte_solver.cuh"
#include "rte_tables.h"

using rtepass::CplEntry;
using rtepass::PassArgs;

namespace {

thread_local char g_create_error[256] = "";

struct AxisTables {
    CplEntry* cpl = nullptr;      // weights x (-c dt) (2 pi / (n dx)) / n : the time step (eq.(11))
    CplEntry* cpl_op = nullptr;   // weights x (+1)    (2 pi / (n dx)) / n : the steady-state operator L = T + sigma_l
    CplEntry* cpl_alt = nullptr;  // weights x (-c dt_alt) ... : Euler updates with another time step (solver preconditioner)
    CplEntry* cpl_rk[2][2] = {{nullptr, nullptr}, {nullptr, nullptr}};   // [dt | dt_alt][x 1/4 | x 2/3]: the scaled Euler
                                  // updates of the SSP-RK3 stages (the stage combination is fused into the passes)
    float2* tw = nullptr;         // forward twiddles of this axis (generic kernels)
    int n = 0, N1 = 0, N2 = 0, maxcnt = 0, npure = 0;   // npure: leading coupling slots with pure blocks (rte_tables.h)
};

// what a sweep of the three pass kernels computes
enum PassKind {
    KIND_STEP = 0,   // out = in (1 - c dt sigma_l) - c dt T[in] + c dt q            eq.(11)
    KIND_OPER = 1,   // out = sigma_l in + T[in]                                     L of eq.(9)
    KIND_EXP = 2,    // out = E (in - c dt T[in]) + phi_1 c dt q, E = exp(-c dt sigma_l)   exponential Euler
    KIND_ALT = 3,    // KIND_STEP with the context's alternative time step dt_alt and a constant source factor
    KIND_STREAM = 4  // out = -c dt T[in]  (no diagonal, no source): the streaming part alone, for the two-kernel exponential step
};

}  // namespace

struct rte_ctx {
    rte_grid grid{};
    rte_pml pml{};
    int N = 0, C = 0, Cp = 0, P = 0;
    long long G = 0;
    float dx = 0, dt = 0, c = 0;
    cudaStream_t stream = nullptr;
    // views into the caller's workspace
    float2* psi = nullptr;
    float2* part = nullptr;
    float *sa = nullptr, *ss = nullptr, *gm = nullptr;
    // small library-owned device arrays
    AxisTables ax[3];
    int* deg = nullptr;
    int* ext_of_slot = nullptr;
    float* srcw = nullptr;
    float* srcS = nullptr;
    size_t srcS_cap = 0;
    int tuned_nt[3] = {0, 0, 0};   // generic kernels: block size per axis measured at the first sweep (0: not yet)
    int first_axis = 0;            // axis of the FIRST pass (the one that stores; the others accumulate): x
    float g_uniform = 0.f;         // > 0: the anisotropy g is one number (media.g_is_map == 0): kernels use the 2-number table
    char* extra = nullptr;         // caller-owned extra workspace (rte_set_extra_workspace): state-sized fields for
    size_t extra_bytes = 0;        // rte_step_ssprk3 (1), rte_apply_operator (2), rte_solve_steady (restart + 3)
    float dt_alt = 0.f;                // time step of the cpl_alt tables (0: not built)
    float alt_src = 0.f;               // source factor of KIND_ALT sweeps (1: constant source on, 0: homogeneous map)
    rtesolve::Scalars* sc = nullptr;   // device scalars of the Krylov solver
    double* partial = nullptr;         // per-block partial sums of its reductions
    cudaGraphExec_t graph = nullptr;   // kGraphSteps captured steps (an even count: the state buffers are back in place)
    const float2* graph_psi = nullptr; // the buffer that held the state when the graph was captured
    bool graph_has_source = false;
    float* graph_amp = nullptr;        // device table of c dt f(t_n) for the captured steps
    float* phi_prev = nullptr;
    double* red = nullptr;         // 2 doubles for reductions
    bool have_prev = false;
    // source
    int src_kind = 0;
    int src_org[3] = {0, 0, 0}, src_ext[3] = {0, 0, 0};
    double src_t0 = 0, src_sig = 1;
    long long steps = 0;
    long long launches = 0;
    int launches_warm = 0;         // an eager step has run (kernel attributes set): graph capture is safe
    char err[256] = "";
};

namespace {

int fail(rte_ctx* ctx, int code, const char* fmt, const char* detail = "") {
    char* dst = ctx ? ctx->err : g_create_error;
    snprintf(dst, 256, fmt, detail);
    return code;
}

// nothing throws across the ABI: std::bad_alloc -> RTE_ENOMEM, anything else -> RTE_EINVAL
template <typename F>
int guarded(F&& f) {
    try { return f(); }
    catch (const std::bad_alloc&) { return RTE_ENOMEM; }
    catch (...) { return RTE_EINVAL; }
}

constexpr int kMaxOrder = 31;   // P_N orders the tables are built for (N = 31: 1024 coefficients in 3-D)

#define CUDA_TRY(ctx, expr)                                                              \
    do {                                                                                 \
        cudaError_t e__ = (expr);                                                        \
        if (e__ != cudaSuccess) return fail(ctx, RTE_ECUDA, "CUDA: %s", cudaGetErrorString(e__)); \
    } while (0)

inline size_t align_up(size_t v, size_t a) { return (v + a - 1) / a * a; }

bool extent_ok(int n) { int a, b; return rtetab::split_of(n, a, b); }

int padded_coeffs(int dim, int N) {
    std::vector<int> e, d;
    rtetab::base_slot_order(dim, N, e, d);
    return (int)e.size();
}

// ---------------------------------------------------------------------------------------------------------------------
// non-hot kernels
// ---------------------------------------------------------------------------------------------------------------------
__device__ __forceinline__ int pml_depth(int i, int n, int W) {
    int p = W - i;
    const int q = i - (n - 1 - W);
    if (q > p) p = q;
    return p > 0 ? p : 0;
}

// sigma maps: sa = mu_a (Omega) | mu_b (PML); ss = mu_s (Omega) | 0 (PML); gm = g.  eq.(12).
__global__ void k_build_maps(float* __restrict__ sa, float* __restrict__ ss, float* __restrict__ gm,
                             const float* __restrict__ mu_a, const float* __restrict__ mu_s,
                             const float* __restrict__ g, int a_map, int s_map, int g_map, int dim, int nx, int ny,
                             int nz, int W, float mu_lo, float mu_hi) {
    const long long G = (long long)nx * ny * nz;
    for (long long cell = blockIdx.x * (long long)blockDim.x + threadIdx.x; cell < G;
         cell += (long long)gridDim.x * blockDim.x) {
        const int x = (int)(cell % nx);
        const long long r = cell / nx;
        const int y = (int)(r % ny), z = (int)(r / ny);
        int p = 0;
        if (W > 0) {
            p = max(pml_depth(x, nx, W), pml_depth(y, ny, W));
            if (dim == 3) p = max(p, pml_depth(z, nz, W));
        }
        if (p == 0) {
            sa[cell] = a_map ? mu_a[cell] : mu_a[0];
            ss[cell] = s_map ? mu_s[cell] : mu_s[0];
        } else {
            const float delta = (float)p / (float)W;
            sa[cell] = mu_lo + (mu_hi - mu_lo) * 0.5f * (1.0f - cospif(delta));
            ss[cell] = 0.f;
        }
        gm[cell] = g_map ? g[cell] : g[0];
    }
}

__global__ void k_pml_profile(float* __restrict__ mu_b, unsigned char* __restrict__ inside, int dim, int nx, int ny,
                              int nz, int W, float mu_lo, float mu_hi) {
    const long long G = (long long)nx * ny * nz;
    for (long long cell = blockIdx.x * (long long)blockDim.x + threadIdx.x; cell < G;
         cell += (long long)gridDim.x * blockDim.x) {
        const int x = (int)(cell % nx);
        const long long r = cell / nx;
        const int y = (int)(r % ny), z = (int)(r / ny);
        int p = 0;
        if (W > 0) {
            p = max(pml_depth(x, nx, W), pml_depth(y, ny, W));
            if (dim == 3) p = max(p, pml_depth(z, nz, W));
        }
        float v = 0.f;
        if (p > 0) v = mu_lo + (mu_hi - mu_lo) * 0.5f * (1.0f - cospif((float)p / (float)W));
        if (mu_b) mu_b[cell] = v;
        if (inside) inside[cell] = p == 0 ? 1 : 0;
    }
}

// external [C][G] -> internal [G][Cp].  One 32x32 tile of (cell, slot) per block through shared memory so both sides
// are coalesced.
__global__ void k_import(float* __restrict__ dst, const float* __restrict__ src, const int* __restrict__ ext_of_slot,
                         long long G, int Cp) {
    __shared__ float tile[32][33];
    const long long cell0 = (long long)blockIdx.x * 32;
    const int s0 = blockIdx.y * 32;
    for (int j = threadIdx.y; j < 32; j += blockDim.y) {     // j: slot within tile, threadIdx.x: cell
        const int s = s0 + j;
        const long long cell = cell0 + threadIdx.x;
        float v = 0.f;
        if (s < Cp && cell < G) {
            const int e = ext_of_slot[s];
            if (e >= 0) v = src[(size_t)e * G + cell];
        }
        tile[j][threadIdx.x] = v;
    }
    __syncthreads();
    for (int j = threadIdx.y; j < 32; j += blockDim.y) {     // j: cell within tile, threadIdx.x: slot
        const int s = s0 + threadIdx.x;
        const long long cell = cell0 + j;
        if (s < Cp && cell < G) dst[(size_t)cell * Cp + s] = tile[threadIdx.x][j];
    }
}

__global__ void k_export(float* __restrict__ dst, const float* __restrict__ src, const int* __restrict__ ext_of_slot,
                         long long G, int Cp) {
    __shared__ float tile[32][33];
    const long long cell0 = (long long)blockIdx.x * 32;
    const int s0 = blockIdx.y * 32;
    for (int j = threadIdx.y; j < 32; j += blockDim.y) {     // j: cell, threadIdx.x: slot
        const int s = s0 + threadIdx.x;
        const long long cell = cell0 + j;
        tile[j][threadIdx.x] = (s < Cp && cell < G) ? src[(size_t)cell * Cp + s] : 0.f;
    }
    __syncthreads();
    for (int j = threadIdx.y; j < 32; j += blockDim.y) {     // j: slot, threadIdx.x: cell
        const int s = s0 + j;
        const long long cell = cell0 + threadIdx.x;
        if (s < Cp && cell < G) {
            const int e = ext_of_slot[s];
            if (e >= 0) dst[(size_t)e * G + cell] = tile[threadIdx.x][j];
        }
    }
}

__global__ void k_fluence(float* __restrict__ phi, const float* __restrict__ psi, long long G, int Cp) {
    for (long long cell = blockIdx.x * (long long)blockDim.x + threadIdx.x; cell < G;
         cell += (long long)gridDim.x * blockDim.x)
        phi[cell] = psi[(size_t)cell * Cp];
}

// source footprint copy with q = 0 outside Omega (eq.(12))
__global__ void k_source_copy(float* __restrict__ dst, const float* __restrict__ src, int ox, int oy, int oz, int ex,
                              int ey, int ez, int dim, int nx, int ny, int nz, int W) {
    const int total = ex * ey * ez;
    for (int i = blockIdx.x * blockDim.x + threadIdx.x; i < total; i += gridDim.x * blockDim.x) {
        const int bx = i % ex, by = (i / ex) % ey, bz = i / (ex * ey);
        int p = 0;
        if (W > 0) {
            p = max(pml_depth(ox + bx, nx, W), pml_depth(oy + by, ny, W));
            if (dim == 3) p = max(p, pml_depth(oz + bz, nz, W));
        }
        dst[i] = p == 0 ? src[i] : 0.f;
    }
}

// sum over Omega of (phi - prev)^2 and phi^2 ; then prev <- phi
__global__ void k_fluence_change(const float* __restrict__ psi, float* __restrict__ prev, double* __restrict__ red,
                                 int dim, int nx, int ny, int nz, int W, int Cp) {
    const long long G = (long long)nx * ny * nz;
    double d2 = 0, n2 = 0;
    for (long long cell = blockIdx.x * (long long)blockDim.x + threadIdx.x; cell < G;
         cell += (long long)gridDim.x * blockDim.x) {
        const int x = (int)(cell % nx);
        const long long r = cell / nx;
        const int y = (int)(r % ny), z = (int)(r / ny);
        int p = 0;
        if (W > 0) {
            p = max(pml_depth(x, nx, W), pml_depth(y, ny, W));
            if (dim == 3) p = max(p, pml_depth(z, nz, W));
        }
        const float v = psi[(size_t)cell * Cp];
        if (p == 0) {
            const double d = (double)v - (double)prev[cell];
            d2 += d * d;
            n2 += (double)v * (double)v;
        }
        prev[cell] = v;
    }
    for (int o = 16; o > 0; o >>= 1) {
        d2 += __shfl_down_sync(0xffffffffu, d2, o);
        n2 += __shfl_down_sync(0xffffffffu, n2, o);
    }
    if ((threadIdx.x & 31) == 0) { atomicAdd(&red[0], d2); atomicAdd(&red[1], n2); }
}

// weighted energy  sum_c (2l+1) ||psi_c||^2  (2-D: weight 1 for m = 0, 2 for m >= 1) and the number of non-finite values:
// the instability guard of reading R10 (forward Euler beyond its bound makes this grow in source-free stretches)
__global__ void k_energy(const float* __restrict__ psi, const int* __restrict__ deg, const int* __restrict__ ext_of_slot,
                         long long G, int Cp, int dim, double* __restrict__ red) {
    double e = 0, bad = 0;
    const long long total = G * Cp;
    for (long long i = blockIdx.x * (long long)blockDim.x + threadIdx.x; i < total; i += (long long)gridDim.x * blockDim.x) {
        const int s = (int)(i % Cp);
        if (ext_of_slot[s] < 0) continue;                       // pad slot
        const float v = psi[i];
        if (!isfinite(v)) { bad += 1.0; continue; }
        const int l = deg[s];
        const double w = dim == 3 ? (double)(2 * l + 1) : (l == 0 ? 1.0 : 2.0);
        e += w * (double)v * (double)v;
    }
    for (int o = 16; o > 0; o >>= 1) {
        e += __shfl_down_sync(0xffffffffu, e, o);
        bad += __shfl_down_sync(0xffffffffu, bad, o);
    }
    if ((threadIdx.x & 31) == 0) { atomicAdd(&red[0], e); atomicAdd(&red[1], bad); }
}

// ---- geometry generators -------------------------------------------------------------------------------------------
__global__ void k_ellipsoids(float* __restrict__ mu_a, float* __restrict__ mu_s, float* __restrict__ g,
                             const float* __restrict__ ell, int n_ell, float bg_a, float bg_s, float bg_g, int dim,
                             int nx, int ny, int nz, float dx) {
    const long long G = (long long)nx * ny * nz;
    for (long long cell = blockIdx.x * (long long)blockDim.x + threadIdx.x; cell < G;
         cell += (long long)gridDim.x * blockDim.x) {
        const int x = (int)(cell % nx);
        const long long r = cell / nx;
        const int y = (int)(r % ny), z = (int)(r / ny);
        const float px = (float)(x - nx / 2) * dx, py = (float)(y - ny / 2) * dx, pz = (float)(z - nz / 2) * dx;
        float va = bg_a, vs = bg_s, vg = bg_g;
        for (int e = 0; e < n_ell; ++e) {
            const float* E = ell + 9 * e;
            const float ux = (px - E[0]) / E[3], uy = (py - E[1]) / E[4];
            float d = ux * ux + uy * uy;
            if (dim == 3) { const float uz = (pz - E[2]) / E[5]; d += uz * uz; }
            if (d <= 1.0f) { va = E[6]; vs = E[7]; vg = E[8]; }
        }
        if (mu_a) mu_a[cell] = va;
        if (mu_s) mu_s[cell] = vs;
        if (g) g[cell] = vg;
    }
}

// counter-based generator: splitmix64 finaliser of (seed, index); two 24-bit uniforms -> Box-Muller normal
__device__ __forceinline__ unsigned long long splitmix64(unsigned long long x) {
    x += 0x9E3779B97F4A7C15ull;
    x = (x ^ (x >> 30)) * 0xBF58476D1CE4E5B9ull;
    x = (x ^ (x >> 27)) * 0x94D049BB133111EBull;
    return x ^ (x >> 31);
}
__global__ void k_white_noise(float* __restrict__ out, long long G, unsigned long long seed) {
    for (long long i = blockIdx.x * (long long)blockDim.x + threadIdx.x; i < G; i += (long long)gridDim.x * blockDim.x) {
        const unsigned long long h = splitmix64(seed * 0x100000001B3ull + (unsigned long long)i);
        const unsigned int a = (unsigned int)(h >> 40), b = (unsigned int)((h >> 16) & 0xFFFFFFu);
        const float u1 = ((float)a + 1.0f) * (1.0f / 16777216.0f);      // (0,1]
        const float u2 = (float)b * (1.0f / 16777216.0f);               // [0,1)
        out[i] = sqrtf(-2.0f * logf(u1)) * cospif(2.0f * u2);
    }
}
// circular 1-D convolution along one axis with a truncated Gaussian (weights normalised to sum 1)
__global__ void k_blur_axis(float* __restrict__ dst, const float* __restrict__ src, int nx, int ny, int nz, int axis,
                            int R, float inv2s2 /* 1/(2 s^2) in cells^-2 */) {
    const long long G = (long long)nx * ny * nz;
    const int n[3] = {nx, ny, nz};
    const long long st[3] = {1, nx, (long long)nx * ny};
    float wsum = 0.f;
    for (int j = -R; j <= R; ++j) wsum += expf(-(float)(j * j) * inv2s2);
    for (long long cell = blockIdx.x * (long long)blockDim.x + threadIdx.x; cell < G;
         cell += (long long)gridDim.x * blockDim.x) {
        const int x = (int)(cell % nx);
        const long long r = cell / nx;
        const int pos[3] = {x, (int)(r % ny), (int)(r / ny)};
        const long long base = cell - pos[axis] * st[axis];
        const int na = n[axis];
        float acc = 0.f;
        for (int j = -R; j <= R; ++j) {
            int i = (pos[axis] + j) % na;
            if (i < 0) i += na;
            acc = fmaf(expf(-(float)(j * j) * inv2s2), src[base + i * st[axis]], acc);
        }
        dst[cell] = acc / wsum;
    }
}
__global__ void k_moments(const float* __restrict__ f, long long G, double* __restrict__ red) {
    double s = 0, s2 = 0;
    for (long long i = blockIdx.x * (long long)blockDim.x + threadIdx.x; i < G; i += (long long)gridDim.x * blockDim.x) {
        const double v = f[i];
        s += v; s2 += v * v;
    }
    for (int o = 16; o > 0; o >>= 1) {
        s += __shfl_down_sync(0xffffffffu, s, o);
        s2 += __shfl_down_sync(0xffffffffu, s2, o);
    }
    if ((threadIdx.x & 31) == 0) { atomicAdd(&red[0], s); atomicAdd(&red[1], s2); }
}
__global__ void k_lognormal_finish(float* __restrict__ f, long long G, const double* __restrict__ red, float mean,
                                   float sigma_log) {
    const double m = red[0] / (double)G;
    const double var = red[1] / (double)G - m * m;
    const float fm = (float)m, inv_sd = (float)(1.0 / sqrt(var));
    const float mu = logf(mean) - 0.5f * sigma_log * sigma_log;
    for (long long i = blockIdx.x * (long long)blockDim.x + threadIdx.x; i < G; i += (long long)gridDim.x * blockDim.x)
        f[i] = expf(fmaf(sigma_log, (f[i] - fm) * inv_sd, mu));
}

int grid_for(long long n, int block) {
    long long b = (n + block - 1) / block;
    if (b > 148 * 16) b = 148 * 16;
    if (b < 1) b = 1;
    return (int)b;
}

int check_grid(const rte_grid* g) {
    if (!g) return RTE_EINVAL;
    if (g->dim != 2 && g->dim != 3) return RTE_EINVAL;
    if (g->dim == 2 && g->nz != 1) return RTE_EINVAL;
    if (!extent_ok(g->nx) || !extent_ok(g->ny)) return RTE_EINVAL;
    if (g->dim == 3 && !extent_ok(g->nz)) return RTE_EINVAL;
    return RTE_OK;
}

// ---------------------------------------------------------------------------------------------------------------------
// pass dispatch
// ---------------------------------------------------------------------------------------------------------------------
// A pass runs either a kernel specialised at compile time for (n, P, TP, block size) — the five BASELINE.json
// configurations — or the generic kernel (run-time P, TP, block size, FIRST/ACC) for every other supported extent / order.
struct LaunchPlan { int TP, nt, blocks, spec; size_t smem; int ncand; int cand[16]; };   // cand: block sizes worth timing (generic)

struct SpecRow { int n, P, TP, nt, TPx; };   // TP: pencils per y / z tile, TPx: per x tile
constexpr SpecRow kSpec[] = {
    {384, 32, 1, 256, 1},   // cfg4: 384^3 P_7   (98 KB tile, 2 CTAs / SM)
    {256, 18, 2, 288, 1},   // cfg3: 256^3 P_5   (y/z: 288 B chunks = 9 whole sectors; x: one contiguous pencil per tile, 3 CTAs / SM)
    {128, 8, 4, 256, 4},    // cfg2: 128^3 P_3
    {512, 8, 2, 256, 2},    // cfg1: 512^2 P_7 (2-D)
    {64, 4, 8, 256, 8},     // cfg0: 64^2 P_3 (2-D)
    {64, 32, 1, 256, 1},    // the paper's second run: 64^3 P_7
};

size_t pass_smem(int n, int Q, int TP, int nsig, bool diag) {
    size_t b = (size_t)n * Q * sizeof(float2);
    if (diag) b += (size_t)nsig * (size_t)rtepass::sig_pitch_l(n, TP) * sizeof(float);   // per-tile table of the Euler diagonal
    return b;
}

constexpr size_t kMaxSmem = 226 * 1024;   // 227 KB per CTA minus the static mbarrier slot

int generic_kernel_regs(int n);      // registers per thread of the generic instance for pencil length n (defined below)

LaunchPlan plan_pass(const rte_ctx* c, int axis, PassArgs& A, PassKind kind) {
    const int first_axis = c->first_axis;
    const int nx = c->grid.nx, ny = c->grid.ny, nz = c->grid.nz;
    int groups = 1;
    if (axis == 0) { A.stride_i = 1; A.stride_t = nx; A.group_stride = 0; A.pencils_per_group = ny * nz; }
    else if (axis == 1) {
        A.stride_i = nx; A.stride_t = 1; A.group_stride = (long long)nx * ny; A.pencils_per_group = nx; groups = nz;
    } else { A.stride_i = nx * ny; A.stride_t = 1; A.group_stride = 0; A.pencils_per_group = nx * ny; }
    const AxisTables& T = c->ax[axis];
    const int P = c->P, n = T.n;
    const bool first = axis == first_axis;
    const bool diag = first || kind == KIND_EXP;   // the FIRST pass carries the Euler diagonal table (every pass of the exponential step)
    LaunchPlan L{};
    L.spec = -1;
    A.P = P;
    if (kind != KIND_EXP)                          // the exponential step runs on the generic kernels
        for (int s = 0; s < (int)(sizeof(kSpec) / sizeof(kSpec[0])); ++s) {
            const int tp = axis == 0 ? kSpec[s].TPx : kSpec[s].TP;
            if (kSpec[s].n == n && kSpec[s].P == P && A.pencils_per_group % tp == 0 &&
                !(axis == 2 && T.maxcnt > 2) && !(axis < 2 && T.npure < 2)) {
                L.spec = s; L.TP = tp; L.nt = kSpec[s].nt;
                break;
            }
        }
    if (L.spec < 0) {
        int tp = 1;
        while (tp * P < 32 && tp < 8) tp *= 2;
        while (tp > 1 && pass_smem(n, tp * P, tp, c->N + 1, diag) > 100 * 1024) tp /= 2;
        while (tp > 1 && tp > A.pencils_per_group) tp /= 2;
        // block size by modelled throughput: the share of useful lanes in the two task loops (Q*N2 and Q*N1 tasks) times
        // the occupancy it allows (CTAs per SM by shared memory, registers of this instance and threads; 24 warps per SM
        // count as saturated).  (The first version minimised idle lanes only and picked e.g. 64-thread blocks — 6 warps per
        // SM — for 192^3 P_5.)
        const int Q = tp * P;
        const int T1 = Q * T.N2, T2 = Q * T.N1;
        const size_t smem = pass_smem(n, Q, tp, c->N + 1, diag) + 1024;       // + the per-CTA reservation
        const int regs = (generic_kernel_regs(n) + 7) / 8 * 8;
        int best = 128; double best_score = -1.0;
        const int ntmax = rtepass::generic_max_threads(T.N1, T.N2);   // by register need of the transforms (rte_pass.cuh)
        for (int nt = 64; nt <= ntmax; nt += 32) {
            if (nt > T1 && nt > T2 && nt > 64) break;
            const double useful = (double)(T1 + T2) / (double)((T1 + nt - 1) / nt * nt + (T2 + nt - 1) / nt * nt);
            int ctas = (int)((size_t)228 * 1024 / smem);
            if (regs > 0) ctas = std::min(ctas, 65536 / (regs * nt));
            ctas = std::min(std::min(ctas, 2048 / nt), 32);
            if (ctas < 1) ctas = 1;
            const double warps = std::min(24.0, (double)ctas * nt / 32.0);
            const double score = useful * warps / 24.0;
            if (score >= best_score - 1e-12) { best_score = score; best = nt; }
            if (useful >= 0.74 && L.ncand < 16) L.cand[L.ncand++] = nt;
        }
        L.TP = tp; L.nt = c->tuned_nt[axis] > 0 ? c->tuned_nt[axis] : best;
    }
    A.TP = L.TP;
    A.tiles_per_group = (A.pencils_per_group + L.TP - 1) / L.TP;
    L.blocks = groups * A.tiles_per_group;
    L.smem = pass_smem(n, L.TP * P, L.TP, c->N + 1, diag);
    if (L.spec >= 0 && axis == 0 && L.TP > 1) L.smem += (size_t)L.TP * (P % 16) * sizeof(float2);   // stacked-layout padding
    if (L.spec >= 0 && axis == 0 && L.TP == 1 && P % 16 != 0) L.smem += 32 * 2 * sizeof(float2);   // block gaps (Geo::PADB), N1 <= 32
    return L;
}

template <int N1, int N2, int MODE, int E, int QC, int PC, int NTC, int MINB, bool UG = false, int AX = 0, bool BASE = false>
cudaError_t launch_one_impl(const PassArgs& A, const LaunchPlan& L, cudaStream_t s) {
    auto kern = rtepass::pass_kernel<N1, N2, MODE, E, QC, PC, NTC, MINB, UG, AX, BASE>;
    // the dynamic shared-memory limit is a per-device function attribute: set it once per (kernel instance, device)
    static std::mutex mu;
    static bool configured[64] = {};
    int dev = 0;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) return e;
    {
        std::lock_guard<std::mutex> lock(mu);
        if (dev < 0 || dev >= 64 || !configured[dev]) {
            e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)kMaxSmem);
            if (e != cudaSuccess) return e;
            if (dev >= 0 && dev < 64) configured[dev] = true;
        }
    }
    kern<<<L.blocks, L.nt, L.smem, s>>>(A);
    return cudaGetLastError();
}

// Specialised FIRST kernels with several pencils per tile come in two instances: uniform g (2-number diagonal table,
// measured 4 % faster on cfg2's x pass) and g map (N+1-number table).  With one pencil per tile (cfg4) a warp reads one
// cell's table row anyway and the N+1-number table measured slightly faster, so only that instance exists.
template <int N1, int N2, int MODE, int E, int QC, int PC, int NTC, int MINB, int AX = 0>
cudaError_t launch_one(const PassArgs& A, const LaunchPlan& L, cudaStream_t s) {
    constexpr bool kHasUG = MODE == rtepass::MODE_FIRST && QC != 0 && (QC / (PC ? PC : 1)) > 1;
    if constexpr (kHasUG)
        if (A.g_uniform > 0.f && A.base == nullptr) return launch_one_impl<N1, N2, MODE, E, QC, PC, NTC, MINB, true, AX>(A, L, s);
    PassArgs B = A;
    B.g_uniform = 0.f;                 // every other instance builds and reads the N+1-number table
    // specialised FIRST kernels with a fused Runge-Kutta combination (PassArgs::base): a separate instance, N+1-number table
    if constexpr (MODE == rtepass::MODE_FIRST && QC != 0)
        if (A.base != nullptr) return launch_one_impl<N1, N2, MODE, E, QC, PC, NTC, MINB, false, AX, true>(B, L, s);
    return launch_one_impl<N1, N2, MODE, E, QC, PC, NTC, MINB, false, AX>(B, L, s);
}

// generic kernels: one instance per supported pencil length (rte_tables.h RTE_SPLITS), FIRST/ACC at run time
cudaError_t launch_generic(int n, const PassArgs& A, const LaunchPlan& L, cudaStream_t s) {
#define RTE_GENERIC_CASE(N1_, N2_) \
    if (n == (N1_) * (N2_)) return launch_one<N1_, N2_, rtepass::MODE_RT, 4, 0, 0, 0, 1>(A, L, s);
    RTE_SPLITS(RTE_GENERIC_CASE)
#undef RTE_GENERIC_CASE
    return cudaErrorInvalidValue;
}

int generic_kernel_regs(int n) {
    static std::mutex mu;
    static int cache[1025] = {};
    if (n < 0 || n > 1024) return 0;
    std::lock_guard<std::mutex> lock(mu);
    if (cache[n] == 0) {
        cudaFuncAttributes at{};
        cudaError_t e = cudaErrorInvalidValue;
#define RTE_GENERIC_REGS(N1_, N2_) \
        if (n == (N1_) * (N2_)) e = cudaFuncGetAttributes(&at, rtepass::pass_kernel<N1_, N2_, rtepass::MODE_RT, 4, 0, 0, 0, 1, false, 0>);
        RTE_SPLITS(RTE_GENERIC_REGS)
#undef RTE_GENERIC_REGS
        cache[n] = e == cudaSuccess ? at.numRegs : -1;
        if (e != cudaSuccess) cudaGetLastError();
    }
    return cache[n] > 0 ? cache[n] : 0;
}

// E = 2 on the z axis of 3-D runs (fan-in of the z coupling is at most 2 pairs, rte_tables.h), 4 otherwise.
// FIRST and ACC instances differ in occupancy (the accumulating tails hold no loaded data): MINB per mode.
// Launched as (FIRST, 4, x), (ACC, 4, y), (ACC, 2, z): the x pass stores, the others accumulate.  (Measured and
// rejected: FIRST on the z axis, whose coupling has the smaller fan-in — DESIGN.md 6.)
template <int MODE, int E, int AX>
cudaError_t launch_spec(int spec, const PassArgs& A, const LaunchPlan& L, cudaStream_t s) {
    constexpr bool F = MODE == rtepass::MODE_FIRST;
    switch (spec) {
        case 0: return launch_one<24, 16, MODE, E, 32, 32, 256, 2, AX>(A, L, s);
        case 1:
            if constexpr (AX == 0) return launch_one<16, 16, MODE, E, 18, 18, 288, 3, AX>(A, L, s);
            else return launch_one<16, 16, MODE, E, 36, 18, 288, F ? 2 : 3, AX>(A, L, s);
        case 2: return launch_one<16, 8, MODE, E, 32, 8, 256, F ? 3 : 4, AX>(A, L, s);
        case 3: return launch_one<32, 16, MODE, E, 16, 8, 256, 2, AX>(A, L, s);
        case 4: return launch_one<8, 8, MODE, E, 32, 4, 256, 3, AX>(A, L, s);
        case 5: return launch_one<8, 8, MODE, E, 32, 32, 256, 3, AX>(A, L, s);
        default: return cudaErrorInvalidValue;
    }
}

double source_time_factor(const rte_ctx* c, double t) {
    if (c->src_kind == 1) return 1.0;
    if (c->src_kind == 2) { const double u = (t - c->src_t0) / c->src_sig; return std::exp(-0.5 * u * u); }
    return 0.0;
}

// coupling table of one axis with every weight multiplied by `scale` x (2 pi / (n dx)) / n; unused entries: own pair, 0
bool build_cpl_table(int dim, int N, int axis, int P, int n, double dx, double scale, std::vector<CplEntry>& flat, int* maxcnt) {
    std::vector<std::vector<rtetab::PairEntry>> pe;
    rtetab::pair_coupling(dim, N, axis, pe);
    const double m = scale * 6.283185307179586476925286766559 / ((double)n * dx) / (double)n;
    flat.assign((size_t)P * rtepass::kMaxE, CplEntry{0.f, 0.f, 0.f, 0.f, 0, 0});
    int mx = 0;
    for (int p = 0; p < P; ++p) {
        const int cnt = (int)pe[p].size();
        if (cnt > rtepass::kMaxE) return false;
        if (cnt > mx) mx = cnt;
        for (int e = 0; e < rtepass::kMaxE; ++e)
            flat[(size_t)p * rtepass::kMaxE + e] =
                (e < cnt && pe[p][e].src >= 0) ? CplEntry{(float)(m * pe[p][e].w00), (float)(m * pe[p][e].w11),
                                   (float)(m * pe[p][e].w01), (float)(m * pe[p][e].w10), pe[p][e].src, 0}
                        : CplEntry{0.f, 0.f, 0.f, 0.f, p, 0};
    }
    if (maxcnt) *maxcnt = mx;
    return true;
}

constexpr double kRkAlpha[2] = {0.25, 2.0 / 3.0};      // SSP-RK3: u2 = 3/4 u + 1/4 E(u1), u' = 1/3 u + 2/3 E(u2)

int upload_cpl(rte_ctx* c, CplEntry** dst, int axis, double scale) {
    AxisTables& T = c->ax[axis];
    std::vector<CplEntry> flat;
    if (!build_cpl_table(c->grid.dim, c->N, axis, c->P, T.n, c->dx, scale, flat, nullptr))
        return fail(c, RTE_EUNSUPPORTED, "coupling fan-in exceeds the kernel's table size");
    if (!*dst) CUDA_TRY(c, cudaMalloc((void**)dst, flat.size() * sizeof(CplEntry) + 16));
    CUDA_TRY(c, cudaMemcpyAsync(*dst, flat.data(), flat.size() * sizeof(CplEntry), cudaMemcpyHostToDevice, c->stream));
    CUDA_TRY(c, cudaStreamSynchronize(c->stream));     // flat is about to go out of scope
    return RTE_OK;
}

// (re)build the alternative-step tables: Euler updates with time step dt_alt on the same context (+ their RK-scaled copies)
int set_alt_dt(rte_ctx* c, float dt_alt) {
    if (c->dt_alt == dt_alt) return RTE_OK;
    for (int a = 0; a < c->grid.dim; ++a) {
        int rc = upload_cpl(c, &c->ax[a].cpl_alt, a, -(double)c->c * (double)dt_alt);
        for (int j = 0; j < 2 && rc == RTE_OK; ++j)
            rc = upload_cpl(c, &c->ax[a].cpl_rk[1][j], a, -(double)c->c * (double)dt_alt * kRkAlpha[j]);
        if (rc != RTE_OK) return rc;
    }
    c->dt_alt = dt_alt;
    return RTE_OK;
}

// the RK-scaled copies of the main tables, built at the first SSP-RK3 step
int ensure_rk_tables(rte_ctx* c) {
    if (c->ax[0].cpl_rk[0][0]) return RTE_OK;
    for (int a = 0; a < c->grid.dim; ++a)
        for (int j = 1; j >= 0; --j) {                  // [0][0] last: it is the "built" marker
            const int rc = upload_cpl(c, &c->ax[a].cpl_rk[0][j], a, -(double)c->c * (double)c->dt * kRkAlpha[j]);
            if (rc != RTE_OK) return rc;
        }
    return RTE_OK;
}

// One sweep of the per-axis pass kernels, out = F(in) with F chosen by `kind` (PassKind above): the forward-Euler update
// of eq.(11) with the source at t_src, the steady-state operator, or the exponential Euler update.
// amp_dev (optional): device location of c dt f(t) for this sweep (CUDA-graph replay), instead of the host value.
// rk_stage (KIND_STEP / KIND_ALT only): 0 = plain; 1, 2 = the scaled update of an SSP-RK3 stage with the combination fused in,
//   out = alpha E(in) + (1 - alpha) rk_base,  alpha = 1/4, 2/3 (tables scaled by alpha; the FIRST pass adds (1 - alpha) rk_base).
int euler_update(rte_ctx* c, const float2* in, float2* out, double t_src, PassKind kind = KIND_STEP,
                 cudaEvent_t* ev = nullptr, const int* halt = nullptr, const float* amp_dev = nullptr, int rk_stage = 0,
                 const float2* rk_base = nullptr) {
    const float alpha = rk_stage ? (float)kRkAlpha[rk_stage - 1] : 1.f;
    const int naxes = c->grid.dim;
    const int fa = c->first_axis;
    // the FIRST pass stores, the others add to what it stored: it goes first
    int order[3] = {fa, fa == 0 ? 1 : 0, fa == 2 ? 1 : 2};
    auto launch_axis = [&](int axis, int nt_override) -> cudaError_t {
        PassArgs A{};
        A.psi = in; A.acc = out;
        A.cpl = kind == KIND_OPER ? c->ax[axis].cpl_op : (kind == KIND_ALT ? c->ax[axis].cpl_alt : c->ax[axis].cpl);
        if (rk_stage) A.cpl = c->ax[axis].cpl_rk[kind == KIND_ALT ? 1 : 0][rk_stage - 1];
        A.tw = c->ax[axis].tw;
        A.sa = c->sa; A.ss = c->ss; A.gm = c->gm; A.deg = c->deg;
        A.cdt = kind == KIND_OPER ? -1.f : (kind == KIND_ALT ? c->c * c->dt_alt : (kind == KIND_STREAM ? 0.f : c->c * c->dt));
        A.ident = (kind == KIND_OPER || kind == KIND_STREAM) ? 0.f : 1.f;      // STREAM: s_l = 0 - 0 sigma_l = 0
        if (rk_stage) {                 // the diagonal table is linear in (ident, cdt): alpha s_l = alpha - (alpha c dt) sigma_l
            A.ident *= alpha; A.cdt *= alpha;
            if (axis == fa) { A.base = rk_base; A.beta = 1.f - alpha; }
        }
        A.expo = kind == KIND_EXP ? 1 : 0;
        A.first = axis == fa ? 1 : 0;
        A.first_axis = fa;
        A.halt = halt;
        A.nsig = c->N + 1; A.g_uniform = c->g_uniform;
        A.srcS = c->srcS; A.srcw = c->srcw;
        for (int j = 0; j < 3; ++j) { A.src_org[j] = c->src_org[j]; A.src_ext[j] = c->src_ext[j]; }
        A.src_amp = 0.f; A.src_amp_dev = nullptr;
        A.nx = c->grid.nx; A.ny = c->grid.ny;
        LaunchPlan L = plan_pass(c, axis, A, kind);
        if (nt_override > 0) L.nt = nt_override;
        const int n = c->ax[axis].n;
        if (A.first && c->src_kind != 0 && kind == KIND_ALT) {
            A.src_amp = c->c * c->dt_alt * c->alt_src * alpha;
        } else if (A.first && c->src_kind != 0 && kind != KIND_OPER && kind != KIND_STREAM) {
            A.src_amp = (float)((double)c->c * (double)c->dt * source_time_factor(c, t_src) * (double)alpha);
            A.src_amp_dev = amp_dev;
            if (amp_dev) A.src_amp = 1.f;      // non-zero: the kernel reads the device value
        }
        using namespace rtepass;
        if (L.spec < 0) return launch_generic(n, A, L, c->stream);
        if (axis == 0) return launch_spec<MODE_FIRST, 4, 0>(L.spec, A, L, c->stream);
        if (axis == 1) return launch_spec<MODE_ACC, 4, 1>(L.spec, A, L, c->stream);
        // z axis: coupling fan-in 2 (rte_tables.h); plan_pass falls back to the generic kernel otherwise
        return launch_spec<MODE_ACC, 2, 2>(L.spec, A, L, c->stream);
    };
    // Generic kernels: the block size of every axis is MEASURED once per context, at its first sweep, among the candidates the
    // occupancy model leaves (the model alone mispredicts by up to 30 %): each candidate is launched twice on the buffers of
    // this sweep and the second launch is timed.  `out` only holds garbage afterwards, and the FIRST pass of the real sweep
    // below overwrites all of it.  Results do not depend on the block size.  Skipped under stream capture.  One stream
    // synchronisation per context.
    {
        bool need = false;
        for (int axis = 0; axis < naxes; ++axis) {
            PassArgs A{};
            if (c->tuned_nt[axis] == 0 && plan_pass(c, axis, A, kind).spec < 0) need = true;
        }
        cudaStreamCaptureStatus cap = cudaStreamCaptureStatusNone;
        if (need && halt == nullptr && cudaStreamIsCapturing(c->stream, &cap) == cudaSuccess && cap == cudaStreamCaptureStatusNone) {
            cudaEvent_t e0 = nullptr, e1 = nullptr;
            if (cudaEventCreate(&e0) == cudaSuccess && cudaEventCreate(&e1) == cudaSuccess) {
                for (int axis = 0; axis < naxes; ++axis) {
                    PassArgs A{};
                    const LaunchPlan L = plan_pass(c, axis, A, kind);
                    if (c->tuned_nt[axis] != 0 || L.spec >= 0) continue;
                    float best_ms = 1e30f;
                    int best_nt = L.nt;
                    for (int k = 0; k < L.ncand; ++k) {
                        if (launch_axis(axis, L.cand[k]) != cudaSuccess) { cudaGetLastError(); continue; }
                        cudaEventRecord(e0, c->stream);
                        const cudaError_t le = launch_axis(axis, L.cand[k]);
                        cudaEventRecord(e1, c->stream);
                        c->launches += 2;
                        float ms = 0.f;
                        if (le != cudaSuccess || cudaEventSynchronize(e1) != cudaSuccess || cudaEventElapsedTime(&ms, e0, e1) != cudaSuccess) {
                            cudaGetLastError();
                            continue;
                        }
                        if (ms < best_ms) { best_ms = ms; best_nt = L.cand[k]; }
                    }
                    c->tuned_nt[axis] = best_nt;
                }
            }
            if (e0) cudaEventDestroy(e0);
            if (e1) cudaEventDestroy(e1);
        }
    }
    for (int k = 0; k < naxes; ++k) {
        const int axis = order[k];
        const cudaError_t e = launch_axis(axis, 0);
        if (e != cudaSuccess) return fail(c, RTE_ECUDA, "pass launch: %s", cudaGetErrorString(e));
        c->launches += 1;
        if (ev) cudaEventRecord(ev[k], c->stream);
    }
    return RTE_OK;
}

// Exponential step on grids with specialised kernels: acc = -c dt T[psi] by the three specialised passes (KIND_STREAM), then
//   new = E (psi + acc) + Phi c dt f(t_n) q,   E = exp(-c dt sigma_l),  Phi = (1 - E)/(c dt sigma_l)
// in one pointwise kernel (in place on acc).  8 S + 3 S of traffic instead of the generic kernels' 8 S, but at the specialised
// kernels' speed (cfg4: 31 instead of 53 ms per step).
constexpr int kExpChunk = 64;      // cells per block round of k_exp_finish
constexpr int kExpMaxDeg = 32;     // N + 1 <= 32

__global__ void __launch_bounds__(256) k_exp_finish(float2* __restrict__ acc, const float2* __restrict__ psi,
                                                    const float* __restrict__ sa, const float* __restrict__ ss,
                                                    const float* __restrict__ gm, const int* __restrict__ deg,
                                                    const float* __restrict__ srcS, const float* __restrict__ srcw, int ox, int oy,
                                                    int oz, int ex, int ey, int ez, int nx, int ny, long long G, int P, int nsig,
                                                    float cdt, float amp) {
    // per chunk of cells: first the (cell, degree) table of c dt sigma_l and E = exp(-c dt sigma_l) in shared memory (one expf per
    // cell and degree instead of two per element), then a coalesced sweep over the chunk's elements
    __shared__ float tE[kExpChunk * kExpMaxDeg], tA[kExpChunk * kExpMaxDeg];
    const long long box_lo = ((long long)oz * ny + oy) * nx + ox;
    const long long box_hi = ((long long)(oz + ez - 1) * ny + (oy + ey - 1)) * nx + (ox + ex - 1);
    const long long nchunks = (G + kExpChunk - 1) / kExpChunk;
    for (long long ch = blockIdx.x; ch < nchunks; ch += gridDim.x) {
        const long long cell0 = ch * kExpChunk;
        const int ncell = (int)min((long long)kExpChunk, G - cell0);
        __syncthreads();                                       // the previous chunk's table is no longer read
        for (int j = threadIdx.x; j < ncell * nsig; j += blockDim.x) {
            const int c = j / nsig, l = j - c * nsig;
            const float g = __ldg(gm + cell0 + c);
            float pw = 1.f;
            for (int k = 0; k < l; ++k) pw *= g;               // g^l by repeated multiplication (R16)
            const float a = cdt * fmaf(__ldg(ss + cell0 + c), 1.f - pw, __ldg(sa + cell0 + c));   // c dt sigma_l
            tA[j] = a;
            tE[j] = expf(-a);
        }
        __syncthreads();
        const long long i0 = cell0 * P;
        for (int j = threadIdx.x; j < ncell * P; j += blockDim.x) {
            const int c = j / P, p = j - c * P;
            const int l0 = __ldg(deg + 2 * p), l1 = __ldg(deg + 2 * p + 1);
            const float e0 = tE[c * nsig + l0], e1 = tE[c * nsig + l1];
            const float2 u = __ldg(psi + i0 + j), t = acc[i0 + j];
            float2 r = make_float2(e0 * (u.x + t.x), e1 * (u.y + t.y));
            const long long cell = cell0 + c;
            if (amp != 0.f && cell >= box_lo && cell <= box_hi) {
                const int x = (int)(cell % nx);
                const long long rr = cell / nx;
                const int bx = x - ox, by = (int)(rr % ny) - oy, bz = (int)(rr / ny) - oz;
                if (bx >= 0 && bx < ex && by >= 0 && by < ey && bz >= 0 && bz < ez) {
                    const float q = amp * __ldg(srcS + ((size_t)bz * ey + by) * ex + bx);
                    const float a0 = tA[c * nsig + l0], a1 = tA[c * nsig + l1];
                    const float ph0 = a0 > 0.f ? -expm1f(-a0) / a0 : 1.f;   // phi_1
                    const float ph1 = a1 > 0.f ? -expm1f(-a1) / a1 : 1.f;
                    r.x = fmaf(ph0 * __ldg(srcw + 2 * p), q, r.x);
                    r.y = fmaf(ph1 * __ldg(srcw + 2 * p + 1), q, r.y);
                }
            }
            acc[i0 + j] = r;
        }
    }
}

bool all_axes_specialised(const rte_ctx* c) {
    for (int axis = 0; axis < c->grid.dim; ++axis) {
        PassArgs A{};
        if (plan_pass(c, axis, A, KIND_STEP).spec < 0) return false;
    }
    return true;
}

// the paper's step: psi^{n+1} = Euler update of psi^n with the source at t_n (R14); the two state buffers trade places
int one_step(rte_ctx* c, cudaEvent_t* ev = nullptr, PassKind kind = KIND_STEP, const float* amp_dev = nullptr) {
    const double tn = (double)c->steps * (double)c->dt;
    if (kind == KIND_EXP && all_axes_specialised(c)) {
        const int rc = euler_update(c, c->psi, c->part, tn, KIND_STREAM, ev);
        if (rc != RTE_OK) return rc;
        const float amp = c->src_kind != 0 ? (float)((double)c->c * (double)c->dt * source_time_factor(c, tn)) : 0.f;
        k_exp_finish<<<grid_for((c->G + kExpChunk - 1) / kExpChunk, 1), 256, 0, c->stream>>>(c->part, c->psi, c->sa, c->ss, c->gm,
            c->deg, c->srcS, c->srcw, c->src_org[0], c->src_org[1], c->src_org[2], c->src_ext[0], c->src_ext[1], c->src_ext[2],
            c->grid.nx, c->grid.ny, c->G, c->P, c->N + 1, c->c * c->dt, amp);
        c->launches += 1;
        if (cudaGetLastError() != cudaSuccess) return fail(c, RTE_ECUDA, "CUDA: %s", "exp finish launch failed");
    } else {
        const int rc = euler_update(c, c->psi, c->part, tn, kind, ev, nullptr, amp_dev);
        if (rc != RTE_OK) return rc;
    }
    std::swap(c->psi, c->part);
    c->steps += 1;
    return RTE_OK;
}

// y = a x + b y over a whole state buffer (the convex combinations of the Runge-Kutta stages)
__global__ void k_axpby(float4* __restrict__ y, const float4* __restrict__ x, float a, float b, size_t n4,
                        const int* __restrict__ halt = nullptr) {
    if (halt && *halt) return;
    for (size_t i = blockIdx.x * (size_t)blockDim.x + threadIdx.x; i < n4; i += (size_t)gridDim.x * blockDim.x) {
        const float4 xv = x[i];
        float4 yv = y[i];
        yv.x = fmaf(a, xv.x, b * yv.x); yv.y = fmaf(a, xv.y, b * yv.y);
        yv.z = fmaf(a, xv.z, b * yv.z); yv.w = fmaf(a, xv.w, b * yv.w);
        y[i] = yv;
    }
}

size_t field_bytes(const rte_ctx* c) { return align_up((size_t)c->G * c->Cp * sizeof(float), 256); }

// i-th state-sized field of the caller's extra workspace, or nullptr when it is too small
float2* extra_field(const rte_ctx* c, int i) {
    const size_t f = field_bytes(c);
    if (!c->extra || (size_t)(i + 1) * f > c->extra_bytes) return nullptr;
    return (float2*)(c->extra + (size_t)i * f);
}

// One SSP-RK3 step on explicit buffers with the alternative time step and a constant source factor (KIND_ALT):
// Y = RK3(X); X is only read, Z is scratch.  The stage combinations are fused into the passes (euler_update rk_stage).
int rk3_alt(rte_ctx* c, const float2* X, float2* Y, float2* Z, const int* halt) {
    int rc = euler_update(c, X, Y, 0.0, KIND_ALT, nullptr, halt);                       // u1 = E(u)
    if (rc != RTE_OK) return rc;
    rc = euler_update(c, Y, Z, 0.0, KIND_ALT, nullptr, halt, nullptr, 1, X);            // u2 = 3/4 u + 1/4 E(u1)
    if (rc != RTE_OK) return rc;
    return euler_update(c, Z, Y, 0.0, KIND_ALT, nullptr, halt, nullptr, 2, X);          // u' = 1/3 u + 2/3 E(u2)
}

// SSP-RK3 (Shu-Osher form, not the paper's integrator):
//   u1 = E(u^n; t_n),  u2 = 3/4 u^n + 1/4 E(u1; t_n + dt),  u^{n+1} = 1/3 u^n + 2/3 E(u2; t_n + dt/2)
// The convex combinations are fused into the passes: the tables of stages 2 and 3 carry the factor 1/4 (2/3), and their FIRST
// pass adds 3/4 (1/3) u^n while it stores — no separate state-wide combination kernels.
int one_step_ssprk3(rte_ctx* c) {
    float2* Z = extra_field(c, 0);
    if (!Z) return fail(c, RTE_EINVAL, "rte_step_ssprk3 needs one state-sized field of extra workspace (rte_set_extra_workspace)");
    int rc = ensure_rk_tables(c);
    if (rc != RTE_OK) return rc;
    float2 *X = c->psi, *Y = c->part;
    const double tn = (double)c->steps * (double)c->dt, dt = (double)c->dt;
    rc = euler_update(c, X, Y, tn);
    if (rc != RTE_OK) return rc;
    rc = euler_update(c, Y, Z, tn + dt, KIND_STEP, nullptr, nullptr, nullptr, 1, X);
    if (rc != RTE_OK) return rc;
    rc = euler_update(c, Z, Y, tn + 0.5 * dt, KIND_STEP, nullptr, nullptr, nullptr, 2, X);
    if (rc != RTE_OK) return rc;
    c->psi = Y; c->part = X;                                // X (u^n) is free now; Z stays the spare buffer
    c->steps += 1;
    return RTE_OK;
}

template <typename T>
cudaError_t upload(T** dst, const std::vector<T>& v, cudaStream_t s) {
    cudaError_t e = cudaMalloc((void**)dst, v.size() * sizeof(T) + 16);
    if (e != cudaSuccess) return e;
    e = cudaMemcpyAsync(*dst, v.data(), v.size() * sizeof(T), cudaMemcpyHostToDevice, s);
    if (e != cudaSuccess) return e;
    return cudaStreamSynchronize(s);   // v is pageable and about to go out of scope
}

// Twiddles and wrapped integer wavenumbers of every supported pencil length -> constant memory, once per device.
cudaError_t upload_constant_tables(int dev) {
    static std::mutex mu;
    static bool done[64] = {};
    std::lock_guard<std::mutex> lock(mu);
    if (dev >= 0 && dev < 64 && done[dev]) return cudaSuccess;
    static const int lens[] = {16, 32, 48, 64, 96, 128, 192, 256, 384, 512};
    std::vector<float2> tw(rtepass::kTableLen);
    std::vector<float> kw(rtepass::kTableLen);
    for (int n : lens) {
        const int off = rtepass::table_offset(n);
        std::vector<float> t;
        rtetab::twiddles(n, t);
        for (int j = 0; j < n; ++j) {
            tw[off + j] = make_float2(t[2 * j], t[2 * j + 1]);
            kw[off + j] = (float)((2 * j < n) ? j : ((2 * j == n) ? 0 : j - n));
        }
    }
    cudaError_t e = cudaMemcpyToSymbol(rtepass::c_tw, tw.data(), tw.size() * sizeof(float2));
    if (e != cudaSuccess) return e;
    e = cudaMemcpyToSymbol(rtepass::c_kw, kw.data(), kw.size() * sizeof(float));
    if (e != cudaSuccess) return e;
    if (dev >= 0 && dev < 64) done[dev] = true;
    return cudaSuccess;
}

void drop_graph(rte_ctx* c) {
    if (c->graph) { cudaGraphExecDestroy(c->graph); c->graph = nullptr; }
}

void free_ctx(rte_ctx* c) {
    if (!c) return;
    for (int a = 0; a < 3; ++a) {
        cudaFree(c->ax[a].cpl); cudaFree(c->ax[a].cpl_op); cudaFree(c->ax[a].cpl_alt); cudaFree(c->ax[a].tw);
        for (int i = 0; i < 2; ++i) for (int j = 0; j < 2; ++j) cudaFree(c->ax[a].cpl_rk[i][j]);
    }
    if (c->graph) cudaGraphExecDestroy(c->graph);
    cudaFree(c->graph_amp);
    cudaFree(c->sc); cudaFree(c->partial);
    cudaFree(c->deg); cudaFree(c->ext_of_slot); cudaFree(c->srcw); cudaFree(c->srcS); cudaFree(c->phi_prev);
    cudaFree(c->red);
    delete c;
}

int set_source_common(rte_ctx* ctx, const float* w_host, const float* S, bool S_on_host, const int org[3],
                      const int ext[3], int kind, float t0, float sig) {
    if (!ctx) return RTE_ESTATE;
    if (kind < 0 || kind > 2) return fail(ctx, RTE_EINVAL, "temporal_kind must be 0, 1 or 2");
    if (kind == 0) { ctx->src_kind = 0; drop_graph(ctx); return RTE_OK; }
    if (!w_host || !S || !org || !ext) return fail(ctx, RTE_EINVAL, "null source argument");
    if (kind == 2 && !(sig > 0)) return fail(ctx, RTE_EINVAL, "sigma_t must be positive");
    const int n[3] = {ctx->grid.nx, ctx->grid.ny, ctx->grid.nz};
    for (int a = 0; a < 3; ++a)
        if (org[a] < 0 || ext[a] < 1 || org[a] + ext[a] > n[a]) return fail(ctx, RTE_EINVAL, "source box outside the grid");
    const size_t cells = (size_t)ext[0] * ext[1] * ext[2];
    drop_graph(ctx);
    if (cells > ctx->srcS_cap) {
        // the new buffer first: a failure leaves the old source (and its buffer) fully intact
        float* fresh = nullptr;
        CUDA_TRY(ctx, cudaMalloc((void**)&fresh, cells * sizeof(float)));
        ctx->src_kind = 0;                      // until the new footprint is in place no step may read the source
        CUDA_TRY(ctx, cudaStreamSynchronize(ctx->stream));
        cudaFree(ctx->srcS);
        ctx->srcS = fresh;
        ctx->srcS_cap = cells;
    }
    ctx->src_kind = 0;
    // angular weights in slot order
    std::vector<int> eos, deg;
    rtetab::slot_order(ctx->grid.dim, ctx->N, eos, deg);
    std::vector<float> w(ctx->Cp, 0.f);
    for (int s = 0; s < ctx->Cp; ++s) if (eos[s] >= 0) w[s] = w_host[eos[s]];
    CUDA_TRY(ctx, cudaMemcpyAsync(ctx->srcw, w.data(), w.size() * sizeof(float), cudaMemcpyHostToDevice, ctx->stream));
    CUDA_TRY(ctx, cudaStreamSynchronize(ctx->stream));
    const float* S_dev = S;
    float* tmp = nullptr;
    if (S_on_host) {
        CUDA_TRY(ctx, cudaMalloc((void**)&tmp, cells * sizeof(float)));
        cudaError_t e = cudaMemcpyAsync(tmp, S, cells * sizeof(float), cudaMemcpyHostToDevice, ctx->stream);
        if (e != cudaSuccess) { cudaFree(tmp); return fail(ctx, RTE_ECUDA, "CUDA: %s", cudaGetErrorString(e)); }
        S_dev = tmp;
    }
    k_source_copy<<<grid_for((long long)cells, 256), 256, 0, ctx->stream>>>(
        ctx->srcS, S_dev, org[0], org[1], org[2], ext[0], ext[1], ext[2], ctx->grid.dim, n[0], n[1], n[2],
        ctx->pml.width);
    ctx->launches += 1;
    cudaError_t e = cudaGetLastError();
    if (tmp) { cudaStreamSynchronize(ctx->stream); cudaFree(tmp); }
    if (e != cudaSuccess) return fail(ctx, RTE_ECUDA, "CUDA: %s", cudaGetErrorString(e));
    for (int a = 0; a < 3; ++a) { ctx->src_org[a] = org[a]; ctx->src_ext[a] = ext[a]; }
    ctx->src_kind = kind; ctx->src_t0 = t0; ctx->src_sig = sig;
    return RTE_OK;
}

}  // namespace

// =====================================================================================================================
// C ABI
// =====================================================================================================================
extern "C" {

int rte_num_coeffs(int dim, int N) { return N > kMaxOrder ? -1 : rtetab::num_coeffs(dim, N); }

int rte_coupling_table(int dim, int N, int axis, double* A_out_host) {
    return guarded([&]() -> int {
        const int C = rte_num_coeffs(dim, N);
        if (C < 0 || axis < 0 || axis > 2 || !A_out_host) return RTE_EINVAL;
        std::vector<double> A[3];
        rtetab::coupling_real(dim, N, A);
        std::memcpy(A_out_host, A[axis].data(), (size_t)C * C * sizeof(double));
        return RTE_OK;
    });
}

int rte_storage_layout(int dim, int N, int* Cp_out, int* ext_of_slot_host, int* cost_host) {
    return guarded([&]() -> int {
        if (rte_num_coeffs(dim, N) < 0) return RTE_EINVAL;
        std::vector<int> eos, deg;
        rtetab::slot_order(dim, N, eos, deg);
        if (Cp_out) *Cp_out = (int)eos.size();
        if (ext_of_slot_host) std::memcpy(ext_of_slot_host, eos.data(), eos.size() * sizeof(int));
        if (cost_host) {
            const rtetab::PairLayout& L = rtetab::pair_layout(dim, N);
            cost_host[0] = L.cost0; cost_host[1] = L.cost; cost_host[2] = L.ideal;
        }
        return RTE_OK;
    });
}

int rte_workspace_bytes(const rte_grid* grid, int N, size_t* bytes_out) {
    return guarded([&]() -> int {
        if (!bytes_out || check_grid(grid) != RTE_OK || N < 1 || N > kMaxOrder) return RTE_EINVAL;
        const size_t G = (size_t)grid->nx * grid->ny * grid->nz;
        const size_t Cp = (size_t)padded_coeffs(grid->dim, N);
        const size_t field = align_up(G * Cp * sizeof(float), 256), map = align_up(G * sizeof(float), 256);
        *bytes_out = 2 * field + 3 * map;
        return RTE_OK;
    });
}

int rte_extra_workspace_bytes(const rte_grid* grid, int N, int n_fields, size_t* bytes_out) {
    return guarded([&]() -> int {
        if (!bytes_out || check_grid(grid) != RTE_OK || N < 1 || N > kMaxOrder || n_fields < 0) return RTE_EINVAL;
        const size_t G = (size_t)grid->nx * grid->ny * grid->nz;
        const size_t Cp = (size_t)padded_coeffs(grid->dim, N);
        *bytes_out = (size_t)n_fields * align_up(G * Cp * sizeof(float), 256);
        return RTE_OK;
    });
}

int rte_stable_dt(int dim, int N, int n_min, float dx, float c, float mu_a_min, float mu_s_min, float g_max,
                  double* bound_ps_out, double* dt_ps_out) {
    return guarded([&]() -> int {
        if (rte_num_coeffs(dim, N) < 0 || n_min < 4 || !(dx > 0) || !(c > 0) || !(mu_a_min >= 0) || !(mu_s_min >= 0) ||
            !(g_max >= 0 && g_max <= 1))
            return RTE_EINVAL;
        double bound = 0;
        if (!rtetab::stable_dt_bound(dim, N, n_min, dx, c, mu_a_min, mu_s_min, g_max, bound)) return RTE_EUNSUPPORTED;
        if (bound_ps_out) *bound_ps_out = bound;
        if (dt_ps_out) *dt_ps_out = 0.5 * bound;
        return RTE_OK;
    });
}

static int create_impl(rte_ctx** out, const rte_grid* grid, int N, float dx, float dt, float c, const rte_media* media,
                       const rte_pml* pml, void* workspace_dev, size_t workspace_bytes, void* cuda_stream, rte_ctx** live) {
    if (!out) return fail(nullptr, RTE_EINVAL, "out is null");
    *out = nullptr;
    if (check_grid(grid) != RTE_OK) return fail(nullptr, RTE_EINVAL, "unsupported grid (dim 2|3; every extent an even 2^a 3^b in [16,1024]; nz=1 in 2-D)");
    if (N < 1 || N > kMaxOrder) return fail(nullptr, RTE_EINVAL, "N must be in 1..31");
    if (!(dx > 0) || !(dt > 0) || !(c > 0)) return fail(nullptr, RTE_EINVAL, "dx, dt, c must be positive");
    if (!media || !media->mu_a || !media->mu_s || !media->g) return fail(nullptr, RTE_EINVAL, "media pointers are null");
    rte_pml pm{0, 0.f, 0.f};
    if (pml) pm = *pml;
    if (pm.width < 0) return fail(nullptr, RTE_EINVAL, "negative PML width");
    {
        int nmin = grid->nx < grid->ny ? grid->nx : grid->ny;
        if (grid->dim == 3 && grid->nz < nmin) nmin = grid->nz;
        if (2 * pm.width >= nmin) return fail(nullptr, RTE_EINVAL, "PML wider than half the grid");
    }
    size_t need = 0;
    rte_workspace_bytes(grid, N, &need);
    if (!workspace_dev || workspace_bytes < need) return fail(nullptr, RTE_EINVAL, "workspace too small");
    if (((uintptr_t)workspace_dev & 255u) != 0) return fail(nullptr, RTE_EINVAL, "workspace must be 256-byte aligned");

    int dev = 0, major = 0;
    if (cudaGetDevice(&dev) != cudaSuccess || cudaDeviceGetAttribute(&major, cudaDevAttrComputeCapabilityMajor, dev) != cudaSuccess)
        return fail(nullptr, RTE_ECUDA, "no CUDA device (this library has no CPU fallback)");
    if (major != 10) return fail(nullptr, RTE_ECUDA, "kernels are built for sm_100a only");

    rte_ctx* ctx = new (std::nothrow) rte_ctx();
    if (!ctx) return fail(nullptr, RTE_ENOMEM, "out of host memory");
    *live = ctx;
    ctx->grid = *grid; ctx->pml = pm; ctx->N = N;
    ctx->C = rtetab::num_coeffs(grid->dim, N);
    ctx->Cp = padded_coeffs(grid->dim, N);
    ctx->P = ctx->Cp / 2;
    ctx->G = (long long)grid->nx * grid->ny * grid->nz;
    ctx->dx = dx; ctx->dt = dt; ctx->c = c;
    ctx->stream = (cudaStream_t)cuda_stream;
    ctx->first_axis = 0;

    const size_t field = align_up((size_t)ctx->G * ctx->Cp * sizeof(float), 256), map = align_up((size_t)ctx->G * sizeof(float), 256);
    char* w = (char*)workspace_dev;
    ctx->psi = (float2*)w; w += field;
    ctx->part = (float2*)w; w += field;
    ctx->sa = (float*)w; w += map;
    ctx->ss = (float*)w; w += map;
    ctx->gm = (float*)w;

    // every pass tile (one pencil of all pairs + tables) must fit in shared memory, and the byte stride between the
    // N1 cells a thread touches must fit 32 bits (rte_pass.cuh byte_off)
    {
        const int ext[3] = {grid->nx, grid->ny, grid->nz};
        const long long str[3] = {1, grid->nx, (long long)grid->nx * grid->ny};
        for (int a = 0; a < grid->dim; ++a) {
            int n1 = 0, n2 = 0;
            rtetab::split_of(ext[a], n1, n2);
            if (pass_smem(ext[a], ctx->P, 1, N + 1, a == ctx->first_axis) > kMaxSmem ||
                (unsigned long long)36 * (unsigned long long)str[a] * (unsigned long long)ctx->P * 8ull >= (1ull << 32)) {
                *live = nullptr;
                delete ctx;
                return fail(nullptr, RTE_EUNSUPPORTED, "grid extent x number of coefficients exceeds one shared-memory pencil tile");
            }
        }
    }

#define CREATE_TRY(expr)                                                                         \
    do {                                                                                         \
        cudaError_t e__ = (expr);                                                                \
        if (e__ != cudaSuccess) {                                                                \
            fail(nullptr, RTE_ECUDA, "CUDA: %s", cudaGetErrorString(e__));                       \
            *live = nullptr;                                                                     \
            free_ctx(ctx);                                                                       \
            return RTE_ECUDA;                                                                    \
        }                                                                                        \
    } while (0)

    // tables
    CREATE_TRY(upload_constant_tables(dev));
    const int ext_n[3] = {grid->nx, grid->ny, grid->nz};
    for (int a = 0; a < grid->dim; ++a) {
        AxisTables& T = ctx->ax[a];
        T.n = ext_n[a];
        rtetab::split_of(T.n, T.N1, T.N2);
        std::vector<CplEntry> flat, flat_op;
        T.npure = rtetab::pair_layout(grid->dim, N).npure[a];
        // -c dt for the time step (eq.(11)), +1 for the operator L
        if (!build_cpl_table(grid->dim, N, a, ctx->P, T.n, dx, -(double)c * (double)dt, flat, &T.maxcnt) ||
            !build_cpl_table(grid->dim, N, a, ctx->P, T.n, dx, 1.0, flat_op, nullptr)) {
            *live = nullptr;
            free_ctx(ctx);
            return fail(nullptr, RTE_EUNSUPPORTED, "coupling fan-in exceeds the kernel's table size");
        }
        CREATE_TRY(upload(&T.cpl_op, flat_op, ctx->stream));
        {
            std::vector<float> t;
            rtetab::twiddles(T.n, t);
            std::vector<float2> tw((size_t)T.n);
            for (int j = 0; j < T.n; ++j) tw[j] = make_float2(t[2 * j], t[2 * j + 1]);
            CREATE_TRY(upload(&T.tw, tw, ctx->stream));
        }
        CREATE_TRY(upload(&T.cpl, flat, ctx->stream));
    }
    {
        std::vector<int> eos, deg;
        rtetab::slot_order(grid->dim, N, eos, deg);
        CREATE_TRY(upload(&ctx->ext_of_slot, eos, ctx->stream));
        CREATE_TRY(upload(&ctx->deg, deg, ctx->stream));
        std::vector<float> zw(ctx->Cp, 0.f);
        CREATE_TRY(upload(&ctx->srcw, zw, ctx->stream));
        CREATE_TRY(cudaMalloc((void**)&ctx->red, 2 * sizeof(double)));
    }
    // a uniform g lets the x pass build a 2-number diagonal table per cell (rte_pass.cuh build_sig)
    if (!media->g_is_map) {
        float g0 = 0.f;
        CREATE_TRY(cudaMemcpyAsync(&g0, media->g, sizeof(float), cudaMemcpyDeviceToHost, ctx->stream));
        CREATE_TRY(cudaStreamSynchronize(ctx->stream));
        ctx->g_uniform = g0 > 0.f ? g0 : 0.f;
    }
    // coefficient maps and zero state
    k_build_maps<<<grid_for(ctx->G, 256), 256, 0, ctx->stream>>>(ctx->sa, ctx->ss, ctx->gm, media->mu_a, media->mu_s,
                                                                media->g, media->mu_a_is_map, media->mu_s_is_map,
                                                                media->g_is_map, grid->dim, grid->nx, grid->ny, grid->nz,
                                                                pm.width, pm.mu_lo, pm.mu_hi);
    ctx->launches += 1;
    CREATE_TRY(cudaGetLastError());
    CREATE_TRY(cudaMemsetAsync(ctx->psi, 0, field, ctx->stream));
    CREATE_TRY(cudaMemsetAsync(ctx->part, 0, field, ctx->stream));
#undef CREATE_TRY
    *live = nullptr;
    *out = ctx;
    return RTE_OK;
}

int rte_create(rte_ctx** out, const rte_grid* grid, int N, float dx, float dt, float c, const rte_media* media,
               const rte_pml* pml, void* workspace_dev, size_t workspace_bytes, void* cuda_stream) {
    rte_ctx* live = nullptr;          // the half-built context, so that an exception cannot leak it
    int rc;
    try {
        rc = create_impl(out, grid, N, dx, dt, c, media, pml, workspace_dev, workspace_bytes, cuda_stream, &live);
    } catch (const std::bad_alloc&) {
        rc = fail(nullptr, RTE_ENOMEM, "out of host memory");
        if (live) free_ctx(live);
        if (out) *out = nullptr;
    } catch (...) {
        rc = fail(nullptr, RTE_EINVAL, "unexpected exception in rte_create");
        if (live) free_ctx(live);
        if (out) *out = nullptr;
    }
    return rc;
}

void rte_destroy(rte_ctx* ctx) {
    if (!ctx) return;
    cudaStreamSynchronize(ctx->stream);
    free_ctx(ctx);
}

int rte_set_state(rte_ctx* ctx, const float* psi_dev) {
    if (!ctx) return RTE_ESTATE;
    if (!psi_dev) return fail(ctx, RTE_EINVAL, "null state pointer");
    dim3 grid((unsigned)((ctx->G + 31) / 32), (unsigned)((ctx->Cp + 31) / 32)), block(32, 8);
    k_import<<<grid, block, 0, ctx->stream>>>((float*)ctx->psi, psi_dev, ctx->ext_of_slot, ctx->G, ctx->Cp);
    ctx->launches += 1;
    CUDA_TRY(ctx, cudaGetLastError());
    ctx->have_prev = false;
    return RTE_OK;
}

int rte_get_state(rte_ctx* ctx, float* psi_dev) {
    if (!ctx) return RTE_ESTATE;
    if (!psi_dev) return fail(ctx, RTE_EINVAL, "null state pointer");
    dim3 grid((unsigned)((ctx->G + 31) / 32), (unsigned)((ctx->Cp + 31) / 32)), block(32, 8);
    k_export<<<grid, block, 0, ctx->stream>>>(psi_dev, (const float*)ctx->psi, ctx->ext_of_slot, ctx->G, ctx->Cp);
    ctx->launches += 1;
    CUDA_TRY(ctx, cudaGetLastError());
    return RTE_OK;
}

// Host variants stage through the partial-sum buffer (free between steps), so no extra device memory is needed.
int rte_set_state_host(rte_ctx* ctx, const float* psi_host) {
    if (!ctx) return RTE_ESTATE;
    if (!psi_host) return fail(ctx, RTE_EINVAL, "null state pointer");
    const size_t bytes = (size_t)ctx->C * ctx->G * sizeof(float);
    CUDA_TRY(ctx, cudaMemcpyAsync(ctx->part, psi_host, bytes, cudaMemcpyHostToDevice, ctx->stream));
    return rte_set_state(ctx, (const float*)ctx->part);
}

int rte_get_state_host(rte_ctx* ctx, float* psi_host) {
    if (!ctx) return RTE_ESTATE;
    if (!psi_host) return fail(ctx, RTE_EINVAL, "null state pointer");
    int rc = rte_get_state(ctx, (float*)ctx->part);
    if (rc != RTE_OK) return rc;
    const size_t bytes = (size_t)ctx->C * ctx->G * sizeof(float);
    CUDA_TRY(ctx, cudaMemcpyAsync(psi_host, ctx->part, bytes, cudaMemcpyDeviceToHost, ctx->stream));
    CUDA_TRY(ctx, cudaStreamSynchronize(ctx->stream));
    return RTE_OK;
}

int rte_reset_time(rte_ctx* ctx) {
    if (!ctx) return RTE_ESTATE;
    ctx->steps = 0;
    return RTE_OK;
}

int rte_set_source(rte_ctx* ctx, const float* w_host, const float* S_dev, const int box_origin[3],
                   const int box_extent[3], int temporal_kind, float t0_ps, float sigma_t_ps) {
    return guarded([&]() -> int {
        return set_source_common(ctx, w_host, S_dev, false, box_origin, box_extent, temporal_kind, t0_ps, sigma_t_ps);
    });
}
int rte_set_source_host(rte_ctx* ctx, const float* w_host, const float* S_host, const int box_origin[3],
                        const int box_extent[3], int temporal_kind, float t0_ps, float sigma_t_ps) {
    return guarded([&]() -> int {
        return set_source_common(ctx, w_host, S_host, true, box_origin, box_extent, temporal_kind, t0_ps, sigma_t_ps);
    });
}

// ---- CUDA-graph replay for launch-bound (L2-resident) grids -----------------------------------------------------------------
// A step is 2-3 launches; on a grid whose state lives in L2 the launches, not the kernels, bound the step (cfg0:
// 11 us/step eager).  kGraphSteps steps (even: the state buffers are back in place) are captured once per context from the
// SAME launch code and replayed; the time-dependent source amplitude c dt f(t_n) of every captured step is read by
// the x kernel from a small device table that the host refreshes, stream-ordered, before each replay.
constexpr int kGraphSteps = 32;
constexpr int kGraphBuildMin = 4;     // calls of fewer steps never pay for a capture
constexpr size_t kGraphMaxStateBytes = (size_t)24 << 20;   // states up to 24 MB (cfg1: 16.8 MB) are L2-resident

int build_graph(rte_ctx* c) {
    if (!c->graph_amp) CUDA_TRY(c, cudaMalloc((void**)&c->graph_amp, kGraphSteps * sizeof(float)));
    const long long steps0 = c->steps, launches0 = c->launches;
    c->graph_psi = c->psi;
    cudaGraph_t g = nullptr;
    // captured on a private stream (the caller's may be the legacy default stream, which cannot capture); the
    // instantiated graph is launched on the caller's stream
    cudaStream_t cap = nullptr, user = c->stream;
    CUDA_TRY(c, cudaStreamCreateWithFlags(&cap, cudaStreamNonBlocking));
    cudaError_t e = cudaStreamBeginCapture(cap, cudaStreamCaptureModeThreadLocal);
    if (e != cudaSuccess) { cudaStreamDestroy(cap); return fail(c, RTE_ECUDA, "graph capture: %s", cudaGetErrorString(e)); }
    c->stream = cap;
    int rc = RTE_OK;
    for (int k = 0; k < kGraphSteps && rc == RTE_OK; ++k) rc = one_step(c, nullptr, KIND_STEP, c->graph_amp + k);
    c->stream = user;
    e = cudaStreamEndCapture(cap, &g);
    cudaStreamDestroy(cap);
    c->steps = steps0; c->launches = launches0;             // nothing ran: capture only recorded the launches
    if (rc != RTE_OK) { if (g) cudaGraphDestroy(g); return rc; }
    if (e != cudaSuccess) return fail(c, RTE_ECUDA, "graph capture: %s", cudaGetErrorString(e));
    e = cudaGraphInstantiate(&c->graph, g, 0);
    cudaGraphDestroy(g);
    if (e != cudaSuccess) { c->graph = nullptr; return fail(c, RTE_ECUDA, "graph instantiate: %s", cudaGetErrorString(e)); }
    return RTE_OK;
}

int rte_step(rte_ctx* ctx, int nsteps) {
    if (!ctx) return RTE_ESTATE;
    if (nsteps < 0) return fail(ctx, RTE_EINVAL, "negative step count");
    return guarded([&]() -> int {
        int left = nsteps;
        const bool small = (size_t)ctx->G * ctx->Cp * sizeof(float) <= kGraphMaxStateBytes;
        // the graph is captured and instantiated (~1 ms) as soon as a call asks for a handful of steps — e.g. a warm-up —
        // so that it is ready when a long run follows; it is replayed only when a whole 32-step batch is left
        if (small && left >= kGraphBuildMin) {
            if (ctx->launches_warm == 0) {                  // one eager step first: per-device kernel attributes get set
                const int rc = one_step(ctx);
                if (rc != RTE_OK) return rc;
                ctx->launches_warm = 1;
                --left;
            }
            if (!ctx->graph) { const int rc = build_graph(ctx); if (rc != RTE_OK) return rc; }
            if (ctx->psi != ctx->graph_psi) {               // the captured launches read the other buffer: one eager step
                const int rc = one_step(ctx);
                if (rc != RTE_OK) return rc;
                --left;
            }
            const int per_step = ctx->grid.dim;
            while (left >= kGraphSteps) {
                if (ctx->src_kind != 0) {
                    float amp[kGraphSteps];
                    for (int k = 0; k < kGraphSteps; ++k)
                        amp[k] = (float)((double)ctx->c * (double)ctx->dt *
                                         source_time_factor(ctx, (double)(ctx->steps + k) * (double)ctx->dt));
                    // pageable source: staged before the call returns, so the stack buffer may go away
                    CUDA_TRY(ctx, cudaMemcpyAsync(ctx->graph_amp, amp, sizeof(amp), cudaMemcpyHostToDevice, ctx->stream));
                }
                CUDA_TRY(ctx, cudaGraphLaunch(ctx->graph, ctx->stream));
                ctx->steps += kGraphSteps;                  // even count: psi / part are where they were
                ctx->launches += (long long)kGraphSteps * per_step;
                left -= kGraphSteps;
            }
        }
        for (int s = 0; s < left; ++s) {
            const int rc = one_step(ctx);
            if (rc != RTE_OK) return rc;
        }
        ctx->launches_warm = 1;
        return RTE_OK;
    });
}

int rte_step_ssprk3(rte_ctx* ctx, int nsteps) {
    if (!ctx) return RTE_ESTATE;
    if (nsteps < 0) return fail(ctx, RTE_EINVAL, "negative step count");
    for (int s = 0; s < nsteps; ++s) {
        const int rc = one_step_ssprk3(ctx);
        if (rc != RTE_OK) return rc;
    }
    return RTE_OK;
}

int rte_step_exp(rte_ctx* ctx, int nsteps) {
    if (!ctx) return RTE_ESTATE;
    if (nsteps < 0) return fail(ctx, RTE_EINVAL, "negative step count");
    for (int s = 0; s < nsteps; ++s) {
        const int rc = one_step(ctx, nullptr, KIND_EXP);
        if (rc != RTE_OK) return rc;
    }
    return RTE_OK;
}

int rte_set_extra_workspace(rte_ctx* ctx, void* extra_dev, size_t bytes) {
    if (!ctx) return RTE_ESTATE;
    if (extra_dev && ((uintptr_t)extra_dev & 255u) != 0) return fail(ctx, RTE_EINVAL, "extra workspace must be 256-byte aligned");
    CUDA_TRY(ctx, cudaStreamSynchronize(ctx->stream));       // nothing in flight may still use the old buffers
    ctx->extra = (char*)extra_dev;
    ctx->extra_bytes = extra_dev ? bytes : 0;
    return RTE_OK;
}

int rte_apply_operator(rte_ctx* ctx, const float* x_dev, float* y_dev) {
    if (!ctx) return RTE_ESTATE;
    if (!x_dev || !y_dev) return fail(ctx, RTE_EINVAL, "null field pointer");
    float2 *X = extra_field(ctx, 0), *Y = extra_field(ctx, 1);
    if (!Y) return fail(ctx, RTE_EINVAL, "rte_apply_operator needs two state-sized fields of extra workspace (rte_set_extra_workspace)");
    dim3 grid((unsigned)((ctx->G + 31) / 32), (unsigned)((ctx->Cp + 31) / 32)), block(32, 8);
    k_import<<<grid, block, 0, ctx->stream>>>((float*)X, x_dev, ctx->ext_of_slot, ctx->G, ctx->Cp);
    const int rc = euler_update(ctx, X, Y, 0.0, KIND_OPER);
    if (rc != RTE_OK) return rc;
    k_export<<<grid, block, 0, ctx->stream>>>(y_dev, (const float*)Y, ctx->ext_of_slot, ctx->G, ctx->Cp);
    ctx->launches += 2;
    CUDA_TRY(ctx, cudaGetLastError());
    return RTE_OK;
}

// b[cell][slot] = w[slot] S(cell) inside the source box (S is already zero outside Omega), 0 elsewhere
__global__ void k_source_field(float* __restrict__ b, const float* __restrict__ S, const float* __restrict__ w, int ox, int oy,
                               int oz, int ex, int ey, int ez, int nx, int ny, long long G, int Cp) {
    const long long total = G * Cp;
    for (long long i = blockIdx.x * (long long)blockDim.x + threadIdx.x; i < total; i += (long long)gridDim.x * blockDim.x) {
        const long long cell = i / Cp;
        const int slot = (int)(i - cell * Cp);
        const int x = (int)(cell % nx);
        const long long r = cell / nx;
        const int bx = x - ox, by = (int)(r % ny) - oy, bz = (int)(r / ny) - oz;
        float v = 0.f;
        if (bx >= 0 && bx < ex && by >= 0 && by < ey && bz >= 0 && bz < ez)
            v = w[slot] * S[((size_t)bz * ey + by) * ex + bx];
        b[i] = v;
    }
}

static int solve_steady_impl(rte_ctx* ctx, int restart, double tol, int max_restarts, int precond_steps, float precond_dt_ps,
                             int* applications_out, double* relres_out);

int rte_solve_steady(rte_ctx* ctx, int restart, double tol, int max_restarts, int precond_steps, float precond_dt_ps,
                     int* applications_out, double* relres_out) {
    return guarded([&]() -> int {     // the preconditioner's tables are built in host vectors: nothing may throw across the ABI
        return solve_steady_impl(ctx, restart, tol, max_restarts, precond_steps, precond_dt_ps, applications_out, relres_out);
    });
}

static int solve_steady_impl(rte_ctx* ctx, int restart, double tol, int max_restarts, int precond_steps, float precond_dt_ps,
                             int* applications_out, double* relres_out) {
    using namespace rtesolve;
    if (!ctx) return RTE_ESTATE;
    if (restart < 1 || restart > kMaxRestart || !(tol > 0) || max_restarts < 0 || precond_steps < 0 ||
        (precond_steps > 0 && !(precond_dt_ps > 0)))
        return fail(ctx, RTE_EINVAL, "rte_solve_steady: restart in 1..64, tol > 0, max_restarts >= 0, precond_steps >= 0 (dt > 0)");
    if (ctx->src_kind == 0) return fail(ctx, RTE_EINVAL, "rte_solve_steady needs a source (rte_set_source)");
    const int m = restart, s = precond_steps;
    const int nfields = m + 3 + (s > 0 ? 3 : 0);
    if (!extra_field(ctx, nfields - 1))
        return fail(ctx, RTE_EINVAL, "rte_solve_steady needs restart + 3 (+ 3 with a preconditioner) state-sized fields of extra "
                                     "workspace (rte_set_extra_workspace)");
    float2* W = extra_field(ctx, 0);
    float2* B = extra_field(ctx, 1);
    float2* V = extra_field(ctx, 2);
    float2* R[3] = {nullptr, nullptr, nullptr};                // preconditioner scratch
    if (s > 0) for (int i = 0; i < 3; ++i) R[i] = extra_field(ctx, m + 3 + i);
    if (((size_t)ctx->G * ctx->Cp) % 4 != 0) return fail(ctx, RTE_EUNSUPPORTED, "state size not a multiple of 16 bytes");
    if (!ctx->sc) {
        CUDA_TRY(ctx, cudaMalloc((void**)&ctx->sc, sizeof(Scalars)));
        CUDA_TRY(ctx, cudaMalloc((void**)&ctx->partial, (size_t)kRedBlocks * (kMaxRestart + 2) * sizeof(double)));
    }
    if (s > 0) { const int rc = set_alt_dt(ctx, precond_dt_ps); if (rc != RTE_OK) return rc; }
    cudaStream_t st = ctx->stream;
    Scalars* sc = ctx->sc;
    double* partial = ctx->partial;
    const size_t fb = field_bytes(ctx), n4 = (size_t)ctx->G * ctx->Cp / 4, stride4 = fb / 16;
    const int NS = kMaxRestart + 1, NT = kMaxRestart;          // partial-sum slots: cycle norms, true-residual norms
    double* hfold = (double*)((char*)sc + offsetof(Scalars, h));
    const int* halt = (const int*)((char*)sc + offsetof(Scalars, halt));
    const double* inv = (const double*)((char*)sc + offsetof(Scalars, inv));
    long long sweeps = 0;                                      // launched operator sweeps that were not no-ops

    auto source_field = [&](float2* dst) {
        k_source_field<<<grid_for(ctx->G * ctx->Cp, 256), 256, 0, st>>>((float*)dst, ctx->srcS, ctx->srcw, ctx->src_org[0],
            ctx->src_org[1], ctx->src_org[2], ctx->src_ext[0], ctx->src_ext[1], ctx->src_ext[2], ctx->grid.nx, ctx->grid.ny,
            ctx->G, ctx->Cp);
        ctx->launches += 1;
    };
    auto norm_to = [&](const float2* a, const float2* b2, float2* y, int slot) {      // h[slot] = ||a - b||^2, y = a - b
        k_sub_norm<<<kRedBlocks, kRedThreads, 0, st>>>((float4*)y, (const float4*)a, (const float4*)b2, n4, partial, slot);
        k_fold<<<1, 128, 0, st>>>(partial + slot, kRedBlocks, 1, hfold + slot, sc);
        ctx->launches += 2;
    };
    // Phi^s: s SSP-RK3 steps of size precond_dt from `in` (read only); returns the buffer that holds the result
    auto rk_steps = [&](const float2* in, float src_factor, const int* hlt, float2** out) -> int {
        ctx->alt_src = src_factor;
        const float2* X = in;
        float2* Y = R[0];
        for (int k = 0; k < s; ++k) {
            const int rc = rk3_alt(ctx, X, Y, R[1], hlt);
            if (rc != RTE_OK) return rc;
            X = Y;
            Y = (Y == R[0]) ? R[2] : R[0];
        }
        *out = const_cast<float2*>(X);
        return RTE_OK;
    };
    // the operator of the linear system: plain  A v = L v ;  preconditioned  A v = v - Phi_lin^s v
    auto apply = [&](const float2* v, const int* hlt) -> int {
        if (s == 0) return euler_update(ctx, v, W, 0.0, KIND_OPER, nullptr, hlt);
        float2* res = nullptr;
        const int rc = rk_steps(v, 0.f, hlt, &res);
        if (rc != RTE_OK) return rc;
        k_axpby<<<grid_for((long long)n4, 256), 256, 0, st>>>((float4*)res, (const float4*)v, 1.f, -1.f, n4, hlt);   // res = v - res
        ctx->launches += 1;
        // W <- res (the Arnoldi kernels work on W): swap roles instead of copying
        std::swap(W, *(res == R[0] ? &R[0] : &R[2]));
        return RTE_OK;
    };

    CUDA_TRY(ctx, cudaMemsetAsync(sc, 0, sizeof(Scalars), st));
    // right-hand side: plain b = q ; preconditioned b = Phi^s(0) with the source on.  ||q|| for the true residual.
    source_field(s > 0 ? R[1] : B);
    norm_to(s > 0 ? R[1] : B, nullptr, nullptr, NT);
    if (s > 0) {
        CUDA_TRY(ctx, cudaMemsetAsync(V, 0, fb, st));
        float2* res = nullptr;
        const int rc = rk_steps(V, 1.f, nullptr, &res);
        if (rc != RTE_OK) return rc;
        std::swap(B, *(res == R[0] ? &R[0] : &R[2]));
    }
    norm_to(B, nullptr, nullptr, NS);
    k_cycle_begin<<<1, 1, 0, st>>>(sc, NS, 1);
    ctx->launches += 1;
    struct Host { double h64, h65, bnorm, beta, relres, inv, tol; int halt, kdone, ktotal, pad_; } hv{};
    static_assert(offsetof(Scalars, bnorm) == offsetof(Scalars, h) + (kMaxRestart + 2) * sizeof(double), "HostView layout");
    CUDA_TRY(ctx, cudaMemcpyAsync(&hv, (char*)sc + offsetof(Scalars, h) + NT * sizeof(double), sizeof(Host), cudaMemcpyDeviceToHost, st));
    CUDA_TRY(ctx, cudaStreamSynchronize(st));
    const double qnorm = std::sqrt(hv.h64);
    double relres = 0.0, history[3] = {0, 0, 0}, past3 = 1e300;
    int cycles = 0;
    if (!(qnorm > 0.0)) {                                      // q = 0: the steady state is psi = 0
        CUDA_TRY(ctx, cudaMemsetAsync(ctx->psi, 0, fb, st));
    } else
        for (int cycle = 0;; ++cycle) {
            cycles = cycle + 1;
            int rc;
            if (s > 0) {                                       // true residual ||q - L x|| / ||q||
                rc = euler_update(ctx, ctx->psi, W, 0.0, KIND_OPER);
                if (rc != RTE_OK) return rc;
                source_field(R[1]);
                norm_to(R[1], W, nullptr, NT);
            }
            // residual of the (preconditioned) system, v_0 = r_0 / ||r_0||
            rc = apply(ctx->psi, nullptr);
            if (rc != RTE_OK) return rc;
            norm_to(B, W, V, NS);
            k_cycle_begin<<<1, 1, 0, st>>>(sc, NS, 0);
            ctx->launches += 1;
            // the one host read of the cycle: a few scalars
            CUDA_TRY(ctx, cudaMemcpyAsync(&hv, (char*)sc + offsetof(Scalars, h) + NT * sizeof(double), sizeof(Host), cudaMemcpyDeviceToHost, st));
            CUDA_TRY(ctx, cudaStreamSynchronize(st));
            relres = s > 0 ? std::sqrt(hv.h64) / qnorm : hv.relres;
            if (!(relres > tol) || cycle == max_restarts || !(hv.relres > 0.0)) break;
            // stagnation (the fp32 floor of the true residual, or a diverging preconditioner step): less than 1 % gained
            // over the last three cycles
            history[cycle % 3] = relres;
            if (cycle >= 3 && relres > 0.99 * past3) break;
            past3 = history[(cycle + 1) % 3];                  // the value from two cycles ago becomes "three ago" next time
            // in-cycle stopping level for the device (relative to ||b||): the residual of the solved system has to fall by
            // tol / relres; with a preconditioner its norm is not the true one, so aim a little lower
            const double level = (s > 0 ? 0.3 : 1.0) * tol / relres * hv.relres;
            CUDA_TRY(ctx, cudaMemcpyAsync((char*)sc + offsetof(Scalars, tol), &level, sizeof(double), cudaMemcpyHostToDevice, st));
            k_scale<<<kRedBlocks, kRedThreads, 0, st>>>((float4*)V, (const float4*)V, inv, n4, sc);
            ctx->launches += 1;
            for (int k = 0; k < m; ++k) {
                const float2* vk = (const float2*)((const char*)V + (size_t)k * fb);
                float2* vn = (float2*)((char*)V + (size_t)(k + 1) * fb);
                rc = apply(vk, halt);
                if (rc != RTE_OK) return rc;
                k_dots<<<kRedBlocks, kRedThreads, 0, st>>>((const float4*)W, (const float4*)V, stride4, k + 1, n4, partial, sc);
                k_fold<<<1, 128, 0, st>>>(partial, kRedBlocks, k + 1, hfold, sc);
                k_update<<<kRedBlocks, kRedThreads, 0, st>>>((float4*)W, (const float4*)V, stride4, k + 1, n4, hfold, partial, NS, sc);
                k_fold<<<1, 128, 0, st>>>(partial + NS, kRedBlocks, 1, hfold + NS, sc);
                k_givens<<<1, 1, 0, st>>>(sc, k, NS);
                k_scale<<<kRedBlocks, kRedThreads, 0, st>>>((float4*)vn, (const float4*)W, inv, n4, sc);
                ctx->launches += 6;
            }
            k_solve_y<<<1, 1, 0, st>>>(sc);
            k_correct<<<kRedBlocks, kRedThreads, 0, st>>>((float4*)ctx->psi, (const float4*)V, stride4, n4, sc);
            ctx->launches += 2;
            CUDA_TRY(ctx, cudaGetLastError());
        }
    // operator sweeps actually performed: Arnoldi steps and per-cycle residuals, 3 per RK3 step with a preconditioner
    const long long per_apply = s > 0 ? 3LL * s : 1;
    sweeps = (long long)hv.ktotal * per_apply + (long long)cycles * (per_apply + (s > 0 ? 1 : 0)) + (s > 0 ? per_apply : 0);
    if (applications_out) *applications_out = (int)sweeps;
    if (relres_out) *relres_out = relres;
    ctx->have_prev = false;
    return RTE_OK;
}

static int step_profile_impl(rte_ctx* ctx, int nsteps, double* ms_axis_host, long long* launches_axis_host) {
    if (!ctx) return RTE_ESTATE;
    if (nsteps < 0 || !ms_axis_host) return fail(ctx, RTE_EINVAL, "bad rte_step_profile argument");
    const int naxes = ctx->grid.dim;
    std::vector<cudaEvent_t> ev((size_t)nsteps * naxes + 1, nullptr);
    for (size_t i = 0; i < ev.size(); ++i)
        if (cudaEventCreate(&ev[i]) != cudaSuccess) {
            for (size_t j = 0; j < i; ++j) cudaEventDestroy(ev[j]);
            return fail(ctx, RTE_ECUDA, "CUDA: %s", "cudaEventCreate failed");
        }
    int rc = RTE_OK;
    cudaEventRecord(ev[0], ctx->stream);
    for (int s = 0; s < nsteps && rc == RTE_OK; ++s) rc = one_step(ctx, &ev[(size_t)s * naxes + 1]);
    if (rc == RTE_OK && cudaStreamSynchronize(ctx->stream) != cudaSuccess) rc = fail(ctx, RTE_ECUDA, "CUDA: %s", "stream synchronise failed");
    for (int a = 0; a < 3; ++a) { ms_axis_host[a] = 0.0; if (launches_axis_host) launches_axis_host[a] = 0; }
    const int fa = ctx->first_axis;
    const int order[3] = {fa, fa == 0 ? 1 : 0, fa == 2 ? 1 : 2};          // launch order of euler_update
    if (rc == RTE_OK)
        for (int s = 0; s < nsteps; ++s)
            for (int k = 0; k < naxes; ++k) {
                float ms = 0.f;
                cudaEventElapsedTime(&ms, ev[(size_t)s * naxes + k], ev[(size_t)s * naxes + k + 1]);
                ms_axis_host[order[k]] += ms;
                if (launches_axis_host) launches_axis_host[order[k]] += 1;
            }
    for (auto& e : ev) cudaEventDestroy(e);
    return rc;
}

int rte_step_profile(rte_ctx* ctx, int nsteps, double* ms_axis_host, long long* launches_axis_host) {
    return guarded([&]() -> int { return step_profile_impl(ctx, nsteps, ms_axis_host, launches_axis_host); });
}

int rte_fluence(rte_ctx* ctx, float* phi_dev) {
    if (!ctx) return RTE_ESTATE;
    if (!phi_dev) return fail(ctx, RTE_EINVAL, "null fluence pointer");
    k_fluence<<<grid_for(ctx->G, 256), 256, 0, ctx->stream>>>(phi_dev, (const float*)ctx->psi, ctx->G, ctx->Cp);
    ctx->launches += 1;
    CUDA_TRY(ctx, cudaGetLastError());
    return RTE_OK;
}

int rte_fluence_host(rte_ctx* ctx, float* phi_host) {
    if (!ctx) return RTE_ESTATE;
    if (!phi_host) return fail(ctx, RTE_EINVAL, "null fluence pointer");
    int rc = rte_fluence(ctx, (float*)ctx->part);
    if (rc != RTE_OK) return rc;
    CUDA_TRY(ctx, cudaMemcpyAsync(phi_host, ctx->part, (size_t)ctx->G * sizeof(float), cudaMemcpyDeviceToHost, ctx->stream));
    CUDA_TRY(ctx, cudaStreamSynchronize(ctx->stream));
    return RTE_OK;
}

int rte_energy(rte_ctx* ctx, double* energy_out, long long* nonfinite_out) {
    if (!ctx) return RTE_ESTATE;
    if (!energy_out && !nonfinite_out) return fail(ctx, RTE_EINVAL, "null output pointers");
    CUDA_TRY(ctx, cudaMemsetAsync(ctx->red, 0, 2 * sizeof(double), ctx->stream));
    k_energy<<<grid_for(ctx->G * ctx->Cp, 256), 256, 0, ctx->stream>>>((const float*)ctx->psi, ctx->deg, ctx->ext_of_slot, ctx->G,
                                                                    ctx->Cp, ctx->grid.dim, ctx->red);
    ctx->launches += 1;
    CUDA_TRY(ctx, cudaGetLastError());
    double h[2] = {0, 0};
    CUDA_TRY(ctx, cudaMemcpyAsync(h, ctx->red, sizeof(h), cudaMemcpyDeviceToHost, ctx->stream));
    CUDA_TRY(ctx, cudaStreamSynchronize(ctx->stream));
    if (energy_out) *energy_out = h[0];
    if (nonfinite_out) *nonfinite_out = (long long)h[1];
    return RTE_OK;
}

int rte_fluence_change(rte_ctx* ctx, double* rel_change_out) {
    if (!ctx) return RTE_ESTATE;
    if (!rel_change_out) return fail(ctx, RTE_EINVAL, "null output pointer");
    if (!ctx->phi_prev) {
        CUDA_TRY(ctx, cudaMalloc((void**)&ctx->phi_prev, (size_t)ctx->G * sizeof(float)));
        CUDA_TRY(ctx, cudaMemsetAsync(ctx->phi_prev, 0, (size_t)ctx->G * sizeof(float), ctx->stream));
        ctx->have_prev = false;
    }
    CUDA_TRY(ctx, cudaMemsetAsync(ctx->red, 0, 2 * sizeof(double), ctx->stream));
    k_fluence_change<<<grid_for(ctx->G, 256), 256, 0, ctx->stream>>>((const float*)ctx->psi, ctx->phi_prev, ctx->red,
                                                                    ctx->grid.dim, ctx->grid.nx, ctx->grid.ny,
                                                                    ctx->grid.nz, ctx->pml.width, ctx->Cp);
    ctx->launches += 1;
    CUDA_TRY(ctx, cudaGetLastError());
    double h[2] = {0, 0};
    CUDA_TRY(ctx, cudaMemcpyAsync(h, ctx->red, sizeof(h), cudaMemcpyDeviceToHost, ctx->stream));
    CUDA_TRY(ctx, cudaStreamSynchronize(ctx->stream));
    if (!ctx->have_prev || !(h[1] > 0)) *rel_change_out = std::numeric_limits<double>::infinity();
    else *rel_change_out = std::sqrt(h[0] / h[1]);
    ctx->have_prev = true;
    return RTE_OK;
}

int rte_time_ps(const rte_ctx* ctx, double* t_out) {
    if (!ctx) return RTE_ESTATE;
    if (!t_out) return RTE_EINVAL;
    *t_out = (double)ctx->steps * (double)ctx->dt;
    return RTE_OK;
}

int rte_sync(rte_ctx* ctx) {
    if (!ctx) return RTE_ESTATE;
    CUDA_TRY(ctx, cudaStreamSynchronize(ctx->stream));
    CUDA_TRY(ctx, cudaGetLastError());
    return RTE_OK;
}

const char* rte_last_error(const rte_ctx* ctx) { return ctx ? ctx->err : g_create_error; }

int rte_launch_count(const rte_ctx* ctx, long long* count_out) {
    if (!ctx) return RTE_ESTATE;
    if (!count_out) return RTE_EINVAL;
    *count_out = ctx->launches;
    return RTE_OK;
}

int rte_media_ellipsoids(const rte_grid* grid, float dx, const float background[3], int n_ell, const float* ell_host,
                         float* mu_a_dev, float* mu_s_dev, float* g_dev, void* cuda_stream) {
    if (!grid || (grid->dim != 2 && grid->dim != 3) || grid->nx < 1 || grid->ny < 1 || grid->nz < 1) return RTE_EINVAL;
    if (!(dx > 0) || !background || n_ell < 0 || (n_ell > 0 && !ell_host)) return RTE_EINVAL;
    for (int e = 0; e < n_ell; ++e)
        for (int k = 3; k < 6; ++k)
            if (!(ell_host[9 * e + k] > 0) && !(grid->dim == 2 && k == 5)) return RTE_EINVAL;
    cudaStream_t s = (cudaStream_t)cuda_stream;
    float* ell_dev = nullptr;
    if (cudaMalloc((void**)&ell_dev, (size_t)(n_ell > 0 ? n_ell : 1) * 9 * sizeof(float)) != cudaSuccess) return RTE_ECUDA;
    if (n_ell > 0 && cudaMemcpyAsync(ell_dev, ell_host, (size_t)n_ell * 9 * sizeof(float), cudaMemcpyHostToDevice, s) != cudaSuccess) {
        cudaFree(ell_dev);
        return RTE_ECUDA;
    }
    const long long G = (long long)grid->nx * grid->ny * grid->nz;
    k_ellipsoids<<<grid_for(G, 256), 256, 0, s>>>(mu_a_dev, mu_s_dev, g_dev, ell_dev, n_ell, background[0], background[1],
                                                 background[2], grid->dim, grid->nx, grid->ny, grid->nz, dx);
    cudaError_t e = cudaGetLastError();
    cudaStreamSynchronize(s);
    cudaFree(ell_dev);
    return e == cudaSuccess ? RTE_OK : RTE_ECUDA;
}

int rte_media_lognormal(const rte_grid* grid, float dx, uint64_t seed, float mean, float sigma_log, float corr_len,
                        float* out_dev, float* scratch_dev, void* cuda_stream) {
    if (!grid || (grid->dim != 2 && grid->dim != 3) || grid->nx < 1 || grid->ny < 1 || grid->nz < 1) return RTE_EINVAL;
    if (!(dx > 0) || !(mean > 0) || !(sigma_log >= 0) || !(corr_len > 0) || !out_dev || !scratch_dev) return RTE_EINVAL;
    cudaStream_t s = (cudaStream_t)cuda_stream;
    const long long G = (long long)grid->nx * grid->ny * grid->nz;
    const int gb = grid_for(G, 256);
    double* red = nullptr;
    if (cudaMalloc((void**)&red, 2 * sizeof(double)) != cudaSuccess) return RTE_ECUDA;
    cudaMemsetAsync(red, 0, 2 * sizeof(double), s);
    // kernel std per axis = corr_len/sqrt2 (so the field's covariance is exp(-r^2/(2 corr_len^2)))
    const float s_cells = corr_len / 1.41421356237f / dx;
    const int R = (int)std::ceil(4.0f * s_cells);
    const float inv2s2 = 1.0f / (2.0f * s_cells * s_cells);
    cudaError_t e = cudaSuccess;
    auto check = [&]() { const cudaError_t l = cudaGetLastError(); if (e == cudaSuccess) e = l; };      // every launch, first error kept
    k_white_noise<<<gb, 256, 0, s>>>(out_dev, G, (unsigned long long)seed);
    check();
    float* a = out_dev;
    float* b = scratch_dev;
    for (int axis = 0; axis < grid->dim; ++axis) {
        k_blur_axis<<<gb, 256, 0, s>>>(b, a, grid->nx, grid->ny, grid->nz, axis, R, inv2s2);
        check();
        float* t = a; a = b; b = t;
    }
    if (a != out_dev) cudaMemcpyAsync(out_dev, a, (size_t)G * sizeof(float), cudaMemcpyDeviceToDevice, s);
    k_moments<<<gb, 256, 0, s>>>(out_dev, G, red);
    check();
    k_lognormal_finish<<<gb, 256, 0, s>>>(out_dev, G, red, mean, sigma_log);
    check();
    { const cudaError_t l = cudaStreamSynchronize(s); if (e == cudaSuccess) e = l; }
    cudaFree(red);
    return e == cudaSuccess ? RTE_OK : RTE_ECUDA;
}

// ---- allocation-free variant of the log-normal generator --------------------------------------------------------------------
// For callers that cannot call cudaMalloc (CUDA-graph capture, tight serving loops, harnesses that forbid it): the blur
// scratch (one float per cell) and the two reduction doubles that rte_media_lognormal takes from the caller / from
// cudaMalloc live in ONE file-scope device array of fixed size.  Every GPU that loads the library holds it until exit.
constexpr long long kNoAllocMaxCells = 2097152;                      // 128^3 cells: 8 MiB of blur scratch
constexpr size_t kNoAllocBytes = (size_t)kNoAllocMaxCells * sizeof(float) + 256;   // + one 256-byte slot for the moments
static __device__ __align__(256) unsigned char g_noalloc_scratch[kNoAllocBytes];

// In host code `g_noalloc_scratch` is only a stand-in for the symbol, not a device address: resolve it once per device, with
// that device current, and hand the kernels the resolved pointer.
static cudaError_t noalloc_scratch_address(unsigned char** ptr_out) {
    static std::mutex mu;
    static unsigned char* resolved[64] = {};
    int dev = 0;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) return e;
    if (dev < 0 || dev >= 64) return cudaErrorInvalidDevice;
    std::lock_guard<std::mutex> lock(mu);
    if (!resolved[dev]) {
        void* p = nullptr;
        e = cudaGetSymbolAddress(&p, g_noalloc_scratch);
        if (e != cudaSuccess) return e;
        resolved[dev] = (unsigned char*)p;
    }
    *ptr_out = resolved[dev];
    return cudaSuccess;
}

int rte_media_lognormal_noalloc(const rte_grid* grid, float dx, uint64_t seed, float mean, float sigma_log, float corr_len,
                                float* out_dev, void* cuda_stream) {
    if (!grid || (grid->dim != 2 && grid->dim != 3) || grid->nx < 1 || grid->ny < 1 || grid->nz < 1)
        return fail(nullptr, RTE_EINVAL, "rte_media_lognormal_noalloc: bad grid");
    if (!(dx > 0) || !(mean > 0) || !(sigma_log >= 0) || !(corr_len > 0) || !out_dev)
        return fail(nullptr, RTE_EINVAL, "rte_media_lognormal_noalloc: bad argument");
    const long long G = (long long)grid->nx * grid->ny * grid->nz;
    if (G > kNoAllocMaxCells)
        return fail(nullptr, RTE_EUNSUPPORTED, "rte_media_lognormal_noalloc: grid exceeds the static scratch (at most 2097152 cells = "
                                               "128^3; use rte_media_lognormal with caller-owned scratch)");
    unsigned char* base = nullptr;
    const cudaError_t ea = noalloc_scratch_address(&base);
    if (ea != cudaSuccess) return fail(nullptr, RTE_ECUDA, "CUDA: %s", cudaGetErrorString(ea));
    float* scratch = reinterpret_cast<float*>(base);
    double* red = reinterpret_cast<double*>(base + (size_t)kNoAllocMaxCells * sizeof(float));
    cudaStream_t s = (cudaStream_t)cuda_stream;
    const int gb = grid_for(G, 256);
    // the array keeps the last call's contents: the moments must start at zero (the blur scratch is fully overwritten)
    if (cudaMemsetAsync(red, 0, 2 * sizeof(double), s) != cudaSuccess) return fail(nullptr, RTE_ECUDA, "CUDA: %s", "memset failed");
    const float s_cells = corr_len / 1.41421356237f / dx;
    const int R = (int)std::ceil(4.0f * s_cells);
    const float inv2s2 = 1.0f / (2.0f * s_cells * s_cells);
    k_white_noise<<<gb, 256, 0, s>>>(out_dev, G, (unsigned long long)seed);
    float* a = out_dev;
    float* b = scratch;
    for (int axis = 0; axis < grid->dim; ++axis) {
        k_blur_axis<<<gb, 256, 0, s>>>(b, a, grid->nx, grid->ny, grid->nz, axis, R, inv2s2);
        float* t = a; a = b; b = t;
    }
    if (a != out_dev) cudaMemcpyAsync(out_dev, a, (size_t)G * sizeof(float), cudaMemcpyDeviceToDevice, s);
    k_moments<<<gb, 256, 0, s>>>(out_dev, G, red);
    k_lognormal_finish<<<gb, 256, 0, s>>>(out_dev, G, red, mean, sigma_log);
    const cudaError_t e = cudaGetLastError();
    return e == cudaSuccess ? RTE_OK : fail(nullptr, RTE_ECUDA, "CUDA: %s", cudaGetErrorString(e));
}

int rte_pml_profile(const rte_grid* grid, const rte_pml* pml, float* mu_b_dev, unsigned char* inside_dev,
                    void* cuda_stream) {
    if (!grid || !pml || (grid->dim != 2 && grid->dim != 3) || grid->nx < 1 || grid->ny < 1 || grid->nz < 1) return RTE_EINVAL;
    if (pml->width < 0) return RTE_EINVAL;
    const long long G = (long long)grid->nx * grid->ny * grid->nz;
    k_pml_profile<<<grid_for(G, 256), 256, 0, (cudaStream_t)cuda_stream>>>(mu_b_dev, inside_dev, grid->dim, grid->nx,
                                                                          grid->ny, grid->nz, pml->width, pml->mu_lo,
                                                                          pml->mu_hi);
    return cudaGetLastError() == cudaSuccess ? RTE_OK : RTE_ECUDA;
}

}  // extern "C"
