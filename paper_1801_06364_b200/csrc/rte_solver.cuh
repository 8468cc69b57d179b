// rte_solver.cuh — device-resident restarted GMRES(m) for the steady state  L psi = q,  L = T + sigma_l  (eq.(9) with
// d/dt = 0; "Krylov subspace iterative methods can then be employed to find a steady-state solution
// through repeated application of the implicit operator": the paper's bottleneck was the host<->device
// traffic of a CPU-side Krylov solver).  SURVEY 8(f1).
//
// Everything lives on the device: the Krylov basis, the Hessenberg matrix, the Givens rotations, the least-squares
// right-hand side and the convergence flag.  The host only enqueues kernels and reads a few scalars per restart cycle
// (the true relative residual, the Arnoldi step count).  Optionally the system is preconditioned by time stepping:
// A = I - Phi^s with Phi one SSP-RK3 step of the same transport operator (rte_lib.cu rte_solve_steady).  No library: dot products, updates and the small dense algebra are the kernels below.
//
// Arnoldi step k (classical Gram-Schmidt, one fused pass each):
//   w = L v_k                               three pass kernels (rte_pass.cuh) with the operator tables
//   h_j = <w, v_j>, j <= k                  k_dots     (per-block partial sums in fp64, fixed order => deterministic)
//                                           k_fold     (one block folds the partials)
//   w -= sum_j h_j v_j ; ||w||^2            k_update   (same two-stage reduction)
//   Givens on column k, residual estimate   k_givens   (one thread; sets the halt flag on convergence / breakdown)
//   v_{k+1} = w / h_{k+1,k}                 k_scale
// Every kernel returns at once when the halt flag is up, so a converged cycle costs (almost) nothing to drain.
#pragma once
#include <cuda_runtime.h>

namespace rtesolve {

constexpr int kMaxRestart = 64;
constexpr int kRedBlocks = 592;        // 4 per SM: partial-sum rows
constexpr int kRedThreads = 256;
constexpr int kChunk = 8;              // basis vectors per sweep of k_dots / k_update

// device-resident scalars of one solve
struct Scalars {
    double H[(kMaxRestart + 1) * kMaxRestart];   // Hessenberg, column k holds h_0k .. h_{k+1,k} (row-major, stride kMaxRestart)
    double cs[kMaxRestart], sn[kMaxRestart];     // Givens rotations
    double g[kMaxRestart + 1];                   // rotated right-hand side; |g[k+1]| = residual norm after step k
    double y[kMaxRestart];                       // least-squares solution of the cycle
    double h[kMaxRestart + 2];                   // folded dot products of the current step (+ norm slot)
    double bnorm, beta, relres, inv;             // ||b||, ||r_0|| of the cycle, residual estimate / ||b||, 1/h_{k+1,k}
    double tol;                                  // in-cycle stopping level of the residual estimate / ||b|| (set by the host per cycle)
    int halt, kdone;                             // halt: stop issuing work; kdone: Arnoldi steps completed in this cycle
    int ktotal, pad_;                            // Arnoldi steps completed in all finished cycles
};


__device__ __forceinline__ double block_sum(double v, double* sh) {
    for (int o = 16; o > 0; o >>= 1) v += __shfl_down_sync(0xffffffffu, v, o);
    const int w = threadIdx.x >> 5, l = threadIdx.x & 31;
    __syncthreads();
    if (l == 0) sh[w] = v;
    __syncthreads();
    double r = 0;
    if (threadIdx.x == 0)
        for (int i = 0; i < (int)(blockDim.x >> 5); ++i) r += sh[i];
    return r;      // valid in thread 0
}

// partial[block][j] = sum over the block's elements of w * V_j, j = 0..cnt-1 (V_j = V + j*stride)
__global__ void __launch_bounds__(kRedThreads) k_dots(const float4* __restrict__ w, const float4* __restrict__ V, size_t stride4,
                                                       int cnt, size_t n4, double* __restrict__ partial, const Scalars* sc) {
    if (sc->halt) return;
    __shared__ double sh[kRedThreads / 32];
    for (int j0 = 0; j0 < cnt; j0 += kChunk) {
        double acc[kChunk];
#pragma unroll
        for (int j = 0; j < kChunk; ++j) acc[j] = 0.0;
        for (size_t i = blockIdx.x * (size_t)blockDim.x + threadIdx.x; i < n4; i += (size_t)gridDim.x * blockDim.x) {
            const float4 a = w[i];
#pragma unroll
            for (int j = 0; j < kChunk; ++j)
                if (j0 + j < cnt) {
                    const float4 b = V[(size_t)(j0 + j) * stride4 + i];
                    acc[j] += (double)a.x * b.x + (double)a.y * b.y + (double)a.z * b.z + (double)a.w * b.w;
                }
        }
#pragma unroll
        for (int j = 0; j < kChunk; ++j)
            if (j0 + j < cnt) {
                const double r = block_sum(acc[j], sh);
                if (threadIdx.x == 0) partial[(size_t)blockIdx.x * (kMaxRestart + 2) + j0 + j] = r;
            }
    }
}

// out[j] = sum over blocks of partial[block][j] in block order (deterministic), j = 0..cnt-1
__global__ void k_fold(const double* __restrict__ partial, int nblk, int cnt, double* __restrict__ out, const Scalars* sc) {
    if (sc->halt) return;
    const int j = threadIdx.x;
    if (j >= cnt) return;
    double s = 0;
    for (int b = 0; b < nblk; ++b) s += partial[(size_t)b * (kMaxRestart + 2) + j];
    out[j] = s;
}

// w -= sum_j h[j] V_j ; partial[block][slot] = block's share of ||w_new||^2
__global__ void __launch_bounds__(kRedThreads) k_update(float4* __restrict__ w, const float4* __restrict__ V, size_t stride4, int cnt,
                                                         size_t n4, const double* __restrict__ h, double* __restrict__ partial, int slot,
                                                         const Scalars* sc) {
    if (sc->halt) return;
    __shared__ double sh[kRedThreads / 32];
    __shared__ float hs[kMaxRestart + 2];
    for (int j = threadIdx.x; j < cnt; j += blockDim.x) hs[j] = (float)h[j];
    __syncthreads();
    double nrm = 0.0;
    for (size_t i = blockIdx.x * (size_t)blockDim.x + threadIdx.x; i < n4; i += (size_t)gridDim.x * blockDim.x) {
        float4 a = w[i];
        for (int j = 0; j < cnt; ++j) {
            const float4 b = V[(size_t)j * stride4 + i];
            const float hj = hs[j];
            a.x = fmaf(-hj, b.x, a.x); a.y = fmaf(-hj, b.y, a.y); a.z = fmaf(-hj, b.z, a.z); a.w = fmaf(-hj, b.w, a.w);
        }
        w[i] = a;
        nrm += (double)a.x * a.x + (double)a.y * a.y + (double)a.z * a.z + (double)a.w * a.w;
    }
    const double r = block_sum(nrm, sh);
    if (threadIdx.x == 0) partial[(size_t)blockIdx.x * (kMaxRestart + 2) + slot] = r;
}

// y = a - b ; partial ||y||^2   (residual r = q - L x); also used with b = nullptr for a plain norm of a
__global__ void __launch_bounds__(kRedThreads) k_sub_norm(float4* __restrict__ y, const float4* __restrict__ a, const float4* __restrict__ b,
                                                           size_t n4, double* __restrict__ partial, int slot) {
    __shared__ double sh[kRedThreads / 32];
    double nrm = 0.0;
    for (size_t i = blockIdx.x * (size_t)blockDim.x + threadIdx.x; i < n4; i += (size_t)gridDim.x * blockDim.x) {
        float4 v = a[i];
        if (b) { const float4 u = b[i]; v.x -= u.x; v.y -= u.y; v.z -= u.z; v.w -= u.w; }
        if (y) y[i] = v;
        nrm += (double)v.x * v.x + (double)v.y * v.y + (double)v.z * v.z + (double)v.w * v.w;
    }
    const double r = block_sum(nrm, sh);
    if (threadIdx.x == 0) partial[(size_t)blockIdx.x * (kMaxRestart + 2) + slot] = r;
}

// y = x * (*scale)
__global__ void k_scale(float4* __restrict__ y, const float4* __restrict__ x, const double* __restrict__ scale, size_t n4,
                        const Scalars* sc) {
    if (sc->halt) return;
    const float s = (float)*scale;
    for (size_t i = blockIdx.x * (size_t)blockDim.x + threadIdx.x; i < n4; i += (size_t)gridDim.x * blockDim.x) {
        float4 v = x[i];
        v.x *= s; v.y *= s; v.z *= s; v.w *= s;
        y[i] = v;
    }
}

// x += sum_j y[j] V_j, j < kdone
__global__ void k_correct(float4* __restrict__ x, const float4* __restrict__ V, size_t stride4, size_t n4, const Scalars* sc) {
    __shared__ float ys[kMaxRestart];
    const int cnt = sc->kdone;
    for (int j = threadIdx.x; j < cnt; j += blockDim.x) ys[j] = (float)sc->y[j];
    __syncthreads();
    if (cnt == 0) return;
    for (size_t i = blockIdx.x * (size_t)blockDim.x + threadIdx.x; i < n4; i += (size_t)gridDim.x * blockDim.x) {
        float4 a = x[i];
        for (int j = 0; j < cnt; ++j) {
            const float4 b = V[(size_t)j * stride4 + i];
            const float yj = ys[j];
            a.x = fmaf(yj, b.x, a.x); a.y = fmaf(yj, b.y, a.y); a.z = fmaf(yj, b.z, a.z); a.w = fmaf(yj, b.w, a.w);
        }
        x[i] = a;
    }
}

// ---- the small dense algebra, one thread --------------------------------------------------------------------------------
// start of a cycle: beta = ||r_0|| from the folded norm in h[slot]; g = (beta, 0, ...); relres = beta / ||b||
__global__ void k_cycle_begin(Scalars* sc, int slot, int first_cycle_sets_bnorm) {
    const double nrm = sqrt(sc->h[slot]);
    if (first_cycle_sets_bnorm) { sc->bnorm = nrm; return; }
    sc->beta = nrm;
    sc->relres = sc->bnorm > 0 ? nrm / sc->bnorm : 0.0;
    for (int i = 0; i <= kMaxRestart; ++i) sc->g[i] = 0.0;
    sc->g[0] = nrm;
    sc->kdone = 0;
    sc->halt = nrm == 0.0 ? 1 : 0;      // the host decides on convergence between cycles and sets the in-cycle level
    sc->inv = nrm > 0 ? 1.0 / nrm : 0.0;
}

// after step k: column k of H = (h_0..h_k, ||w||), rotate, new rotation, residual estimate, 1/h_{k+1,k}
__global__ void k_givens(Scalars* sc, int k, int norm_slot) {
    if (sc->halt) return;
    const int m = kMaxRestart;
    const double hn = sqrt(sc->h[norm_slot]);
    double col[kMaxRestart + 1];
    for (int j = 0; j <= k; ++j) col[j] = sc->h[j];
    for (int j = 0; j < k; ++j) {
        const double a = col[j], b = col[j + 1];
        col[j] = sc->cs[j] * a + sc->sn[j] * b;
        col[j + 1] = -sc->sn[j] * a + sc->cs[j] * b;
    }
    const double a = col[k], d = sqrt(a * a + hn * hn);
    const double c = d > 0 ? a / d : 1.0, s = d > 0 ? hn / d : 0.0;
    sc->cs[k] = c; sc->sn[k] = s;
    col[k] = d;
    for (int j = 0; j <= k; ++j) sc->H[j * m + k] = col[j];
    sc->g[k + 1] = -s * sc->g[k];
    sc->g[k] = c * sc->g[k];
    sc->kdone = k + 1;
    sc->relres = fabs(sc->g[k + 1]) / sc->bnorm;
    // happy breakdown (the Krylov space is exhausted) or converged: stop issuing work
    const bool breakdown = !(hn > 1e-7 * fabs(d));
    sc->inv = breakdown ? 0.0 : 1.0 / hn;
    if (breakdown || sc->relres <= sc->tol) sc->halt = 1;
}

// end of a cycle: back substitution  R y = g  over the kdone completed steps
__global__ void k_solve_y(Scalars* sc) {
    const int m = kMaxRestart, k = sc->kdone;
    for (int i = k - 1; i >= 0; --i) {
        double s = sc->g[i];
        for (int j = i + 1; j < k; ++j) s -= sc->H[i * m + j] * sc->y[j];
        const double d = sc->H[i * m + i];
        sc->y[i] = d != 0.0 ? s / d : 0.0;
    }
    sc->ktotal += k;
    sc->halt = 0;      // the correction and the next cycle's residual must run
}

}  // namespace rtesolve
