// rte_pass.cuh — the per-axis pencil kernel of the P_N pseudospectral RTE step (sm_100a).
//
// One launch handles one axis a of the step (PAPER.md:123-127 re-designed):
//   1. load a tile of TP adjacent pencils (all C coefficients of every cell on the pencil) straight from HBM into
//      registers and do the first factor of DFT_n (N1-point transforms)                     eq.(7)-(8)
//   2. second factor (N2-point), multiply by i k_a / n (Nyquist zeroed), inverse second factor  eq.(10)
//   3. inverse first factor -> D_a psi on the pencil, kept in shared memory
//   4. streaming coupling T_c = sum_c' w^a_{cc'} D_a psi_c' (sparse l+-1, m, m+-1)           eq.(6)/(10)
//      and, depending on MODE:
//        FIRST   partial  = T                                (x pass)
//        MIDDLE  partial += T                                (y pass in 3-D)
//        LAST    psi <- psi - c dt (partial + T + sigma_l psi) + c dt q   (last axis: scattering diagonal eq.(9),
//                PML eq.(12), source, forward Euler eq.(11))
// The coefficient fields are stored cell-major, [cell][P] float2 ("pairs", see rte_tables.h), so a pencil along any
// axis is a sequence of P*8-byte contiguous chunks and one complex FFT differentiates two real fields.
//
// Index conventions inside a tile: i = position along the pencil (0..n-1), t = pencil within the tile (0..TP-1),
// p = pair (0..P-1), q = t*P + p (0..Q-1).  Shared tile: tile[i*Q + q].  n = N1*N2, i = a*N2 + b, k = k1 + N1*k2.
#pragma once
#include "rte_fft.cuh"

namespace rtepass {

constexpr int kMaxE = 4;   // max source pairs per output pair and axis (checked on the host when tables are built)

struct CplEntry { int src; float w00, w01, w10, w11; };

enum { MODE_FIRST = 0, MODE_MIDDLE = 1, MODE_LAST = 2 };

struct PassArgs {
    // fields
    const float2* psi;      // [G][P]
    float2* part;           // [G][P] partial streaming sums
    float2* out;            // LAST: where the new state goes (== psi: in place is safe, tiles are disjoint)
    // tables
    const float2* tw;       // [n] forward twiddles exp(-2 pi i j/n)
    const float* kap;       // [n] k_a[j]/n, Nyquist zeroed
    const CplEntry* cpl;    // [P][kMaxE]
    const int* cpl_cnt;     // [P]
    // epilogue (LAST)
    const float* sa;        // [G] mu_a in Omega, mu_b in the PML
    const float* ss;        // [G] mu_s in Omega, 0 in the PML
    const float* gm;        // [G] g
    const int* deg;         // [2P] degree l of every slot
    float cdt;              // c * dt
    // source (LAST)
    const float* srcS;      // [ext z][ext y][ext x], already zero outside Omega
    const float* srcw;      // [2P] angular weight per slot
    int src_org[3], src_ext[3];
    float src_amp;          // c dt f(t_n); 0 => no source this step
    // geometry of this pass
    int stride_i;           // cell stride along the pencil
    int stride_t;           // cell stride between neighbouring pencils of a tile
    int group_stride;       // cell stride between pencil groups
    int pencils_per_group, tiles_per_group;
    int P, TP;
    int nx, ny;
};

// ---- phase 1: HBM -> registers, first factor forward, -> shared -----------------------------------------------------
template <int N1, int N2>
RTE_HD void phase_fwd1(const PassArgs& A, float2* tile, int base, int valid, int tid, int nt) {
    const int Q = A.TP * A.P;
    for (int task = tid; task < Q * N2; task += nt) {
        const int q = task % Q, b = task / Q;
        const int t = q / A.P, p = q - t * A.P;
        float2 v[N1];
        if (t < valid) {
            const float2* src = A.psi + ((size_t)(base + t * A.stride_t + b * A.stride_i)) * A.P + p;
            const size_t step = (size_t)N2 * A.stride_i * A.P;
#pragma unroll
            for (int a = 0; a < N1; ++a) v[a] = src[a * step];
        } else {
#pragma unroll
            for (int a = 0; a < N1; ++a) v[a] = make_float2(0.f, 0.f);
        }
        rtefft::dft_fwd<N1>(v);
#pragma unroll
        for (int k1 = 0; k1 < N1; ++k1) tile[(k1 * N2 + b) * Q + q] = v[k1];
    }
}

// ---- phase 2: twiddle, second factor forward, i k / n, second factor inverse, conjugate twiddle -----------------------
template <int N1, int N2>
RTE_HD void phase_mid(const PassArgs& A, float2* tile, const float2* tw, const float* kap, int tid, int nt) {
    const int Q = A.TP * A.P;
    for (int task = tid; task < Q * N1; task += nt) {
        const int q = task % Q, k1 = task / Q;
        float2* row = tile + (k1 * N2) * Q + q;
        float2 v[N2];
#pragma unroll
        for (int b = 0; b < N2; ++b) v[b] = row[b * Q];
#pragma unroll
        for (int b = 1; b < N2; ++b) v[b] = rtefft::cmul(v[b], tw[b * k1]);
        rtefft::dft_fwd<N2>(v);
#pragma unroll
        for (int k2 = 0; k2 < N2; ++k2) {
            const float kk = kap[k1 + N1 * k2];
            v[k2] = make_float2(-kk * v[k2].y, kk * v[k2].x);   // * i k
        }
        rtefft::dft_inv<N2>(v);
#pragma unroll
        for (int b = 1; b < N2; ++b) v[b] = rtefft::cmulc(v[b], tw[b * k1]);
#pragma unroll
        for (int b = 0; b < N2; ++b) row[b * Q] = v[b];
    }
}

// ---- phase 3: first factor inverse: shared now holds D_a psi for every (i, q) -----------------------------------------
template <int N1, int N2>
RTE_HD void phase_inv1(const PassArgs& A, float2* tile, int tid, int nt) {
    const int Q = A.TP * A.P;
    for (int task = tid; task < Q * N2; task += nt) {
        const int q = task % Q, b = task / Q;
        float2* col = tile + b * Q + q;
        float2 v[N1];
#pragma unroll
        for (int k1 = 0; k1 < N1; ++k1) v[k1] = col[(k1 * N2) * Q];
        rtefft::dft_inv<N1>(v);
#pragma unroll
        for (int a = 0; a < N1; ++a) col[(a * N2) * Q] = v[a];
    }
}

// ---- phase 4: coupling + accumulate / integrate ---------------------------------------------------------------------
template <int N1, int N2, int MODE>
RTE_HD void phase_out(const PassArgs& A, const float2* tile, int base, int valid, int tid, int nt) {
    const int Q = A.TP * A.P;
    for (int task = tid; task < Q * N2; task += nt) {
        const int q = task % Q, b = task / Q;
        const int t = q / A.P, p = q - t * A.P;
        if (t >= valid) continue;
        // this pair's coupling list
        const int cnt = A.cpl_cnt[p];
        int esrc[kMaxE];
        float w00[kMaxE], w01[kMaxE], w10[kMaxE], w11[kMaxE];
#pragma unroll
        for (int e = 0; e < kMaxE; ++e) {
            const CplEntry ce = A.cpl[p * kMaxE + e];
            esrc[e] = ce.src; w00[e] = ce.w00; w01[e] = ce.w01; w10[e] = ce.w10; w11[e] = ce.w11;
        }
        const int cell0 = base + t * A.stride_t + b * A.stride_i;
        int l0 = 0, l1 = 0, sx = 0, sy = 0, sz = 0;
        float sw0 = 0.f, sw1 = 0.f;
        bool src_on = false;
        if (MODE == MODE_LAST) {
            l0 = A.deg[2 * p]; l1 = A.deg[2 * p + 1];
            src_on = (A.src_amp != 0.f);
            if (src_on) {
                sx = cell0 % A.nx - A.src_org[0];
                const int r = cell0 / A.nx;
                sy = r % A.ny - A.src_org[1];
                sz = r / A.ny - A.src_org[2];
                sw0 = A.srcw[2 * p] * A.src_amp; sw1 = A.srcw[2 * p + 1] * A.src_amp;
            }
        }
#pragma unroll 2
        for (int a = 0; a < N1; ++a) {
            const int i = a * N2 + b;
            const float2* row = tile + i * Q + t * A.P;
            float2 T = make_float2(0.f, 0.f);
#pragma unroll
            for (int e = 0; e < kMaxE; ++e)
                if (e < cnt) {
                    const float2 d = row[esrc[e]];
                    T.x = fmaf(w00[e], d.x, T.x); T.x = fmaf(w01[e], d.y, T.x);
                    T.y = fmaf(w10[e], d.x, T.y); T.y = fmaf(w11[e], d.y, T.y);
                }
            const int cell = cell0 + a * N2 * A.stride_i;
            const size_t gi = (size_t)cell * A.P + p;
            if (MODE == MODE_FIRST) {
                A.part[gi] = T;
            } else if (MODE == MODE_MIDDLE) {
                const float2 pt = A.part[gi];
                A.part[gi] = make_float2(pt.x + T.x, pt.y + T.y);
            } else {
                const float2 ps = A.psi[gi];
                const float2 pt = A.part[gi];
                const float sa = A.sa[cell], ss = A.ss[cell], g = A.gm[cell];
                float g0 = 1.f, g1 = 1.f;
                for (int j = 0; j < l0; ++j) g0 *= g;          // g^l by repeated multiplication (R16)
                for (int j = 0; j < l1; ++j) g1 *= g;
                const float sig0 = fmaf(ss, 1.f - g0, sa), sig1 = fmaf(ss, 1.f - g1, sa);
                float2 r;
                r.x = ps.x - A.cdt * ((pt.x + T.x) + sig0 * ps.x);
                r.y = ps.y - A.cdt * ((pt.y + T.y) + sig1 * ps.y);
                if (src_on) {
                    // offset of this cell inside the source box along the pencil axis
                    const int di = a * N2;
                    int bx = sx, by = sy, bz = sz;
                    if (A.stride_i == 1) bx += di; else if (A.stride_i == A.nx) by += di; else bz += di;
                    if (bx >= 0 && bx < A.src_ext[0] && by >= 0 && by < A.src_ext[1] && bz >= 0 && bz < A.src_ext[2]) {
                        const float S = A.srcS[((size_t)bz * A.src_ext[1] + by) * A.src_ext[0] + bx];
                        r.x = fmaf(sw0, S, r.x); r.y = fmaf(sw1, S, r.y);
                    }
                }
                A.out[gi] = r;
            }
        }
    }
}

#ifdef __CUDACC__
template <int N1, int N2, int MODE>
__global__ void __launch_bounds__(320, 1) pass_kernel(const PassArgs A) {
    extern __shared__ float2 smem[];
    constexpr int n = N1 * N2;
    const int Q = A.TP * A.P;
    float2* tile = smem;
    float2* tw = tile + (size_t)n * Q;
    float* kap = reinterpret_cast<float*>(tw + n);
    const int tid = threadIdx.x, nt = blockDim.x;
    for (int i = tid; i < n; i += nt) { tw[i] = A.tw[i]; kap[i] = A.kap[i]; }
    const int group = blockIdx.x / A.tiles_per_group, tin = blockIdx.x - group * A.tiles_per_group;
    const int valid = min(A.TP, A.pencils_per_group - tin * A.TP);
    const int base = group * A.group_stride + tin * A.TP * A.stride_t;
    phase_fwd1<N1, N2>(A, tile, base, valid, tid, nt);
    __syncthreads();
    phase_mid<N1, N2>(A, tile, tw, kap, tid, nt);
    __syncthreads();
    phase_inv1<N1, N2>(A, tile, tid, nt);
    __syncthreads();
    phase_out<N1, N2, MODE>(A, tile, base, valid, tid, nt);
}
#endif

}  // namespace rtepass
