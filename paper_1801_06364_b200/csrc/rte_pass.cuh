// rte_pass.cuh — the per-axis pencil kernel of the P_N pseudospectral RTE step (sm_100a).
//
// One launch handles one axis a of the step (PAPER.md:123-127 re-designed):
//   1. load a tile of TP adjacent pencils (all coefficients of every cell on the pencil) straight from HBM into
//      registers (N1 loads in flight per thread) and do the first factor of DFT_n      eq.(7)-(8)
//   2. second factor (N2-point), multiply by i k_a / n (Nyquist zeroed), inverse second factor  eq.(10)
//   3. inverse first factor -> D_a psi on the pencil, kept in shared memory
//   4. streaming coupling  -c dt T_c = sum_c' w^a_{cc'} D_a psi_c'  (sparse l+-1, m, m+-1; the weights arrive
//      pre-multiplied by -c dt)                                                        eq.(6)/(10)
//      and, depending on MODE, the running forward-Euler accumulator `acc` (eq.(11)):
//        FIRST   acc  = psi (1 - c dt sigma_l) - c dt T_x + c dt q   (x pass: scattering diagonal eq.(9), PML
//                                                                    eq.(12), source)
//        MIDDLE  acc += -c dt T_y                                    (y pass in 3-D)
//        LAST    psi  = acc - c dt T_a                               (last axis; in place: tiles are disjoint and
//                                                                    every read of a tile precedes its writes)
// The coefficient fields are stored cell-major, [cell][P] float2 ("pairs", see rte_tables.h), so a pencil along any
// axis is a sequence of P*8-byte contiguous chunks and one complex FFT differentiates two real fields.
//
// Index conventions inside a tile: i = position along the pencil (0..n-1), t = pencil within the tile (0..TP-1),
// p = pair (0..P-1), q = t*P + p (0..Q-1).  n = N1*N2, i = a*N2 + b, k = k1 + N1*k2.
// Shared tile: element (i, t, p) lives at tile[i*SI + t*ST + p] with
//   (SI, ST) = (Q, P)             "interleaved": y/z passes and every generic kernel — the global order of a y/z tile
//   (SI, ST) = (P, n*P + pad)     "stacked":     x pass of the specialised kernels — the global order of an x tile
// so that the specialised kernels fill the tile with a few TMA bulk copies (cp.async.bulk, SASS UBLKCP) that complete
// on an mbarrier while the CTA loads its tables; the generic kernels load through registers.
// QC / PC / NTC are compile-time copies of Q, P and the block size (0 = run-time value) so that every shared-memory
// offset of the unrolled transforms folds into an instruction immediate for the configurations that matter.
#pragma once
#include "rte_fft.cuh"

namespace rtepass {

constexpr int kMaxE = 4;   // max source pairs per output pair and axis (checked on the host when tables are built)

// One 2x2 real block of the coupling: T.x += wd0 d.x + ws0 d.y ; T.y += wd1 d.y + ws1 d.x  (wd = diagonal (w00, w11),
// ws = off-diagonal (w01, w10); stored as the two register pairs of the packed FFMA2 form).  Weights already
// multiplied by -c dt * 2 pi / (n_a dx) / n_a (Euler step, wavenumber unit and inverse-DFT normalisation of the axis).
struct alignas(8) CplEntry { float wd0, wd1, ws0, ws1; int src; int pad_; };

enum { MODE_FIRST = 0, MODE_MIDDLE = 1, MODE_LAST = 2 };

struct PassArgs {
    // fields
    const float2* psi;      // [G][P]  state at t_n (input of the transform)
    float2* acc;            // [G][P]  running accumulator of the new state
    float2* out;            // LAST: where the new state goes (== psi)
    // tables (twiddles and wrapped integer wavenumbers live in constant memory, see c_tw / c_kw)
    const CplEntry* cpl;    // [P][kMaxE], unused entries: src = own pair, weights 0
    // diagonal + source (FIRST)
    const float* sa;        // [G] mu_a in Omega, mu_b in the PML
    const float* ss;        // [G] mu_s in Omega, 0 in the PML
    const float* gm;        // [G] g
    const int* deg;         // [2P] degree l of every slot
    float cdt;              // c * dt
    int nsig;               // N + 1 degrees
    const float* srcS;      // [ext z][ext y][ext x], already zero outside Omega
    const float* srcw;      // [2P] angular weight per slot
    int src_org[3], src_ext[3];
    float src_amp;          // c dt f(t_n); 0 => no source this step
    // geometry of this pass (cells)
    int stride_i;           // cell stride along the pencil
    int stride_t;           // cell stride between neighbouring pencils of a tile
    long long group_stride; // cell stride between pencil groups
    int pencils_per_group, tiles_per_group;
    int P, TP;
    int nx, ny;
};

// Supported pencil lengths and where their tables start in the constant arrays.
constexpr int kTableLen = 1728;   // 16+32+48+64+96+128+192+256+384+512
#ifdef __CUDACC__
__host__ __device__
#endif
constexpr int table_offset(int n) {
    return n == 16 ? 0 : n == 32 ? 16 : n == 48 ? 48 : n == 64 ? 96 : n == 96 ? 160 : n == 128 ? 256 : n == 192 ? 384
         : n == 256 ? 576 : n == 384 ? 832 : n == 512 ? 1216 : -1;
}

#ifdef __CUDACC__

// c_tw[table_offset(n) + j] = exp(-2 pi i j / n)  (forward twiddles, eq.(8))
// c_kw[table_offset(n) + j] = j for j < n/2, 0 at j = n/2 (Nyquist, R5), j - n above  (exact in fp32)
// Read with warp-uniform (or nearly uniform) indices through the constant cache, which keeps these table reads off
// the shared-memory pipe that bounds the pass kernels.  Filled once per device by rte_create.
__constant__ float2 c_tw[kTableLen];
__constant__ float c_kw[kTableLen];

// ---- global memory access with explicit state space (keeps LDG/STG instead of generic LD/ST after byte offsets) ------
__device__ __forceinline__ float2 ldg64(const float2* p, unsigned long long byte_offset) {
    float2 v;
    asm volatile("ld.global.v2.f32 {%0,%1}, [%2];" : "=f"(v.x), "=f"(v.y) : "l"(reinterpret_cast<const char*>(p) + byte_offset));
    return v;
}
__device__ __forceinline__ void stg64(float2* p, unsigned long long byte_offset, float2 v) {
    asm volatile("st.global.v2.f32 [%0], {%1,%2};" ::"l"(reinterpret_cast<char*>(p) + byte_offset), "f"(v.x), "f"(v.y) : "memory");
}

// ---- mbarrier + TMA bulk copy (global -> shared) ----------------------------------------------------------------------
__device__ __forceinline__ unsigned smem_u32(const void* p) { return (unsigned)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void mbar_init(unsigned long long* bar, unsigned count) {
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(bar)), "r"(count) : "memory");
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
}
__device__ __forceinline__ void mbar_arrive_expect_tx(unsigned long long* bar, unsigned bytes) {
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(bar)), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_wait(unsigned long long* bar, unsigned parity) {
    asm volatile(
        "{\n"
        ".reg .pred p;\n"
        "WAIT_%=:\n"
        "mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n"
        "@p bra DONE_%=;\n"
        "bra WAIT_%=;\n"
        "DONE_%=:\n"
        "}\n" ::"r"(smem_u32(bar)), "r"(parity) : "memory");
}
__device__ __forceinline__ void tma_load_1d(void* smem_dst, const void* gmem_src, unsigned bytes, unsigned long long* bar) {
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];" ::"r"(smem_u32(smem_dst)),
                 "l"(gmem_src), "r"(bytes), "r"(smem_u32(bar))
                 : "memory");
}

// ---- tile geometry ------------------------------------------------------------------------------------------------------
// STACKED (x pass of a specialised kernel): tile[(t*(n*P + pad) + i*P + p]; otherwise tile[i*Q + t*P + p].
// pad = P mod 16 float2 keeps the lanes of a half-warp (consecutive p, then the next pencil) on distinct banks.
template <int N1, int N2, int QC, int PC, bool STACKED>
struct Geo {
    static constexpr int n = N1 * N2;
    static constexpr int TPC = QC / (PC ? PC : 1);
    static constexpr int pad = (STACKED && TPC > 1) ? (PC % 16) : 0;
    static constexpr int SI = STACKED ? PC : QC;             // 0 when run-time
    static constexpr int ST = STACKED ? n * PC + pad : PC;
    static constexpr int tile_elems = STACKED ? TPC * ST : n * QC;
};

// ---- phase 0 (specialised kernels): the whole psi tile by TMA bulk copies ------------------------------------------------
template <int N1, int N2, int QC, int PC, bool STACKED>
__device__ __forceinline__ void tile_tma_load(const PassArgs& A, float2* tile, long long base, unsigned long long* bar, int tid,
                                              int nt) {
    using G = Geo<N1, N2, QC, PC, STACKED>;
    if (STACKED) {
        // TP whole pencils of n*P*8 contiguous bytes each, issued as 16 KB pieces by different threads
        constexpr unsigned pen_bytes = (unsigned)G::n * PC * 8u;
        constexpr unsigned piece = pen_bytes % 16384u == 0 ? 16384u : (pen_bytes % 4096u == 0 ? 4096u : pen_bytes);
        constexpr int pieces = (int)(pen_bytes / piece);
        for (int j = tid; j < G::TPC * pieces; j += nt) {
            const int t = j / pieces, k = j - t * pieces;
            const char* src = reinterpret_cast<const char*>(A.psi + (base + (long long)t * A.stride_t) * PC) + (size_t)k * piece;
            char* dst = reinterpret_cast<char*>(tile + t * G::ST) + (size_t)k * piece;
            tma_load_1d(dst, src, piece, bar);
        }
    } else {
        // n rows of Q*8 contiguous bytes (neighbouring pencils of a y/z tile are neighbouring cells), issued b-major
        // (i = a*N2 + b); the rows of residue b complete on bar[b], so that the phase-1 columns of residue b can start
        // while the rest of the tile is still in flight
        for (int j = tid; j < G::n; j += nt) {
            const int b = j / N1, a = j - b * N1, i = a * N2 + b;
            tma_load_1d(tile + i * QC, A.psi + (base + (long long)i * A.stride_i) * PC, (unsigned)QC * 8u, bar + b);
        }
    }
}

// tile offset of (i = 0, t, p) for the q-th column
template <typename G, bool STACKED>
__device__ __forceinline__ int col_offset(int q, int P) {
    if (STACKED) { const int t = q / P; return t * G::ST + (q - t * P); }
    return q;
}

// ---- phase 1: first factor forward.  Generic: HBM -> registers -> DFT -> shared.  TMA: in place in shared ------------------
// CF ("couple first", specialised kernels): the streaming coupling is applied HERE, to the transform's input —
//   -c dt T_c = D_a ( sum_c' w^a_{cc'} psi_c' )      (constant weights commute with D_a; R18)
// so a column gathers its <= E source pairs from the freshly loaded tile, and the tail needs no neighbour data at all:
// one shared-memory store and E loads per element become E loads, and the tail runs without any barrier.  The
// gather reads rows that other columns of the same rows overwrite, hence the fence between gather and store: the rows
// of one residue b are owned by one warp (32 % Q == 0) or by one round of the whole CTA (nt % Q == 0).
template <int N1, int N2, int E, int QC, int PC, bool STACKED, bool TMA, bool CF>
__device__ __forceinline__ void phase_fwd1(const PassArgs& A, float2* tile, long long base, int valid, int tid, int nt,
                                           unsigned long long* bar) {
    using G = Geo<N1, N2, QC, PC, STACKED>;
    const int P = PC ? PC : A.P;
    const int Q = QC ? QC : A.TP * P;
    const int SI = G::SI ? G::SI : Q;
    const int ST = G::ST ? G::ST : P;
    const unsigned long long stepB = (unsigned long long)N2 * (unsigned)A.stride_i * (unsigned)P * 8u;
#pragma unroll 1
    for (int task = tid; task < Q * N2; task += nt) {
        const int b = task / Q, q = task - b * Q;
        const int t = q / P, p = q - t * P;
        float2* col = tile + b * SI + t * ST + p;
        float2 v[N1];
        if (CF) {
            const float2* srow[E];
            float2 wd[E], ws[E];
#pragma unroll
            for (int e = 0; e < E; ++e) {
                const CplEntry* ce = A.cpl + p * kMaxE + e;
                srow[e] = tile + b * SI + t * ST + __ldg(&ce->src);
                wd[e] = __ldg(reinterpret_cast<const float2*>(&ce->wd0));
                ws[e] = __ldg(reinterpret_cast<const float2*>(&ce->ws0));
            }
            mbar_wait(bar + (STACKED ? 0 : b), 0);
#pragma unroll
            for (int a = 0; a < N1; ++a) {
                float2 u = make_float2(0.f, 0.f);
#pragma unroll
                for (int e = 0; e < E; ++e) {
                    const float2 d = srow[e][(a * N2) * SI];
                    u = rtefft::cfma_diag(wd[e].x, wd[e].y, d, u);
                    u = rtefft::cfma_swap(ws[e].x, ws[e].y, d, u);
                }
                v[a] = u;
            }
            if (QC && 32 % (QC ? QC : 1) == 0) __syncwarp();
            else __syncthreads();
        } else if (TMA) {
            mbar_wait(bar + (STACKED ? 0 : b), 0);
#pragma unroll
            for (int a = 0; a < N1; ++a) v[a] = col[a * N2 * SI];
        } else {
            if (t < valid) {
                const float2* src = A.psi + (base + (long long)t * A.stride_t + (long long)b * A.stride_i) * P + p;
#pragma unroll
                for (int a = 0; a < N1; ++a) v[a] = ldg64(src, stepB * a);
            } else {
#pragma unroll
                for (int a = 0; a < N1; ++a) v[a] = make_float2(0.f, 0.f);
            }
        }
        rtefft::dft_fwd<N1>(v);
#pragma unroll
        for (int k1 = 0; k1 < N1; ++k1) col[k1 * N2 * SI] = v[k1];
    }
}

// ---- phase 2: twiddle, second factor forward, i k / n, second factor inverse, conjugate twiddle -----------------------
template <int N1, int N2, int QC, int PC, bool STACKED>
__device__ __forceinline__ void phase_mid(const PassArgs& A, float2* tile, int tid, int nt) {
    using G = Geo<N1, N2, QC, PC, STACKED>;
    constexpr int off = table_offset(N1 * N2);
    const int P = PC ? PC : A.P;
    const int Q = QC ? QC : A.TP * P;
    const int SI = G::SI ? G::SI : Q;
#pragma unroll 1
    for (int task = tid; task < Q * N1; task += nt) {
        const int k1 = task / Q, q = task - k1 * Q;
        float2* row = tile + (k1 * N2) * SI + col_offset<G, STACKED>(q, P);
        float2 v[N2], w[N2];
#pragma unroll
        for (int b = 0; b < N2; ++b) v[b] = row[b * SI];
#pragma unroll
        for (int b = 1; b < N2; ++b) { w[b] = c_tw[off + k1 * b]; v[b] = rtefft::cmul(v[b], w[b]); }
        rtefft::dft_fwd<N2>(v);
#pragma unroll
        for (int k2 = 0; k2 < N2; ++k2)
            v[k2] = rtefft::cscale(make_float2(-v[k2].y, v[k2].x), c_kw[off + k1 + N1 * k2]);   // * i * wrapped(k); 2 pi/(n dx)/n is in the weights
        rtefft::dft_inv<N2>(v);
#pragma unroll
        for (int b = 1; b < N2; ++b) v[b] = rtefft::cmulc(v[b], w[b]);
#pragma unroll
        for (int b = 0; b < N2; ++b) row[b * SI] = v[b];
    }
}

// ---- phase 3: first factor inverse: shared now holds D_a psi for every (i, q) -----------------------------------------
template <int N1, int N2, int QC, int PC, bool STACKED>
__device__ __forceinline__ void phase_inv1(const PassArgs& A, float2* tile, int tid, int nt) {
    using G = Geo<N1, N2, QC, PC, STACKED>;
    const int P = PC ? PC : A.P;
    const int Q = QC ? QC : A.TP * P;
    const int SI = G::SI ? G::SI : Q;
#pragma unroll 1
    for (int task = tid; task < Q * N2; task += nt) {
        const int b = task / Q, q = task - b * Q;
        float2* col = tile + b * SI + col_offset<G, STACKED>(q, P);
        float2 v[N1];
#pragma unroll
        for (int k1 = 0; k1 < N1; ++k1) v[k1] = col[(k1 * N2) * SI];
        rtefft::dft_inv<N1>(v);
#pragma unroll
        for (int a = 0; a < N1; ++a) col[(a * N2) * SI] = v[a];
    }
}

// ---- FIRST only: per-tile table of the Euler diagonal  s_l(r) = 1 - c dt sigma_l(r) -----------------------------------
// sigma_l = mu_a + mu_s (1 - g^l) in Omega (eq.(9); g^l by repeated multiplication, R16),
//         = mu_b for every l in the PML, where the maps hold (mu_b, 0, g) (eq.(12)).
// Layout sig[l*(ncell+1) + j], j = t*n + i: conflict-free to build (lanes = cells) and to read (lanes = degrees).
template <int N1, int N2>
__device__ __forceinline__ void build_sig(const PassArgs& A, float* sig, long long base, int valid, int tid, int nt) {
    constexpr int n = N1 * N2;
    const int ncell = n * A.TP;
    for (int j = tid; j < ncell; j += nt) {
        const int t = j / n, i = j - t * n;
        float sa = 0.f, ss = 0.f, g = 0.f;
        if (t < valid) {
            const long long cell = base + (long long)t * A.stride_t + (long long)i * A.stride_i;
            sa = __ldg(A.sa + cell); ss = __ldg(A.ss + cell); g = __ldg(A.gm + cell);
        }
        float pw = 1.f;
        float* dst = sig + j;
        for (int l = 0; l < A.nsig; ++l) {
            *dst = 1.f - A.cdt * fmaf(ss, 1.f - pw, sa);
            pw *= g;
            dst += ncell + 1;
        }
    }
}

// ---- phase 4: coupling + accumulate / integrate ---------------------------------------------------------------------
// FUSED (specialised kernels whose warps own whole rows of the tile, 32 % Q == 0): phase 3 runs here, per warp — the
// columns (b, all q) a warp transforms are exactly the rows its coupling reads, so a __syncwarp replaces the CTA barrier,
// the warps drift apart, and the accumulator loads are issued before the inverse DFT and fly under it.
// CF: the coupling was applied in phase 1; the tail is  acc (+)= IDFT_{N1}(column)  straight from registers.
template <int N1, int N2, int MODE, int E, int QC, int PC, bool STACKED, bool FUSED, bool CF>
__device__ __forceinline__ void tail_task(const PassArgs& A, float2* tile, const float* sig, long long base, int valid,
                                          int task, long long pencil0, float2 (&r)[N1], bool loaded) {
    using G = Geo<N1, N2, QC, PC, STACKED>;
    constexpr int n = N1 * N2;
    const int P = PC ? PC : A.P;
    const int Q = QC ? QC : A.TP * P;
    const int SI = G::SI ? G::SI : Q;
    const int ST = G::ST ? G::ST : P;
    const unsigned long long stepB = (unsigned long long)N2 * (unsigned)A.stride_i * (unsigned)P * 8u;
    {
        const int b = task / Q, q = task - b * Q;
        const int t = q / P, p = q - t * P;
        if (t >= valid) return;
        // this pair's coupling list (unused entries point at the pair itself with zero weights)
        const float2* srow[E];
        float2 wd[E], ws[E];
        if (!CF) {
#pragma unroll
            for (int e = 0; e < E; ++e) {
                const CplEntry* ce = A.cpl + p * kMaxE + e;
                srow[e] = tile + b * SI + t * ST + __ldg(&ce->src);
                wd[e] = __ldg(reinterpret_cast<const float2*>(&ce->wd0));
                ws[e] = __ldg(reinterpret_cast<const float2*>(&ce->ws0));
            }
        }
        const long long gi = (base + (long long)t * A.stride_t + (long long)b * A.stride_i) * P + p;
        const float2* lp = (MODE == MODE_FIRST ? A.psi : A.acc) + gi;
        float2* sp = (MODE == MODE_LAST ? A.out : A.acc) + gi;
        if (!loaded) {
#pragma unroll
            for (int a = 0; a < N1; ++a) r[a] = ldg64(lp, stepB * a);
        }
        float2 v[N1];
        if (FUSED || CF) {
            float2* col = tile + b * SI + t * ST + p;
#pragma unroll
            for (int k1 = 0; k1 < N1; ++k1) v[k1] = col[(k1 * N2) * SI];
            rtefft::dft_inv<N1>(v);
            if (!CF) {
#pragma unroll
                for (int a = 0; a < N1; ++a) col[(a * N2) * SI] = v[a];
                __syncwarp();
            }
        }
        const float* s0 = sig;
        const float* s1 = sig;
        if (MODE == MODE_FIRST) {
            const int ncell1 = n * A.TP + 1;
            s0 = sig + __ldg(A.deg + 2 * p) * ncell1 + t * n + b;
            s1 = sig + __ldg(A.deg + 2 * p + 1) * ncell1 + t * n + b;
        }
#pragma unroll
        for (int a = 0; a < N1; ++a) {
            float2 T = make_float2(0.f, 0.f);
            if (CF) T = v[a];
            else {
#pragma unroll
                for (int e = 0; e < E; ++e) {
                    const float2 d = srow[e][(a * N2) * SI];
                    T = rtefft::cfma_diag(wd[e].x, wd[e].y, d, T);
                    T = rtefft::cfma_swap(ws[e].x, ws[e].y, d, T);
                }
            }
            if (MODE == MODE_FIRST) r[a] = rtefft::cfma_diag(s0[a * N2], s1[a * N2], r[a], T);
            else r[a] = rtefft::cadd(r[a], T);
        }
        if (MODE == MODE_FIRST && A.src_amp != 0.f) {
            // FIRST is the x pass: position along the pencil = x, pencil index = y + ny*z
            const long long pen = pencil0 + t;
            const int by = (int)(pen % A.ny) - A.src_org[1], bz = (int)(pen / A.ny) - A.src_org[2];
            if (by >= 0 && by < A.src_ext[1] && bz >= 0 && bz < A.src_ext[2]) {
                const float sw0 = __ldg(A.srcw + 2 * p) * A.src_amp, sw1 = __ldg(A.srcw + 2 * p + 1) * A.src_amp;
                const float* Srow = A.srcS + ((size_t)bz * A.src_ext[1] + by) * A.src_ext[0];
#pragma unroll
                for (int a = 0; a < N1; ++a) {
                    const int bx = a * N2 + b - A.src_org[0];
                    if (bx >= 0 && bx < A.src_ext[0]) {
                        const float S = __ldg(Srow + bx);
                        r[a].x = fmaf(sw0, S, r[a].x); r[a].y = fmaf(sw1, S, r[a].y);
                    }
                }
            }
        }
#pragma unroll
        for (int a = 0; a < N1; ++a) stg64(sp, stepB * a, r[a]);
    }
}

// the global loads of one tail task (accumulator rows; psi itself in the FIRST pass): issued as early as possible
template <int N1, int N2, int MODE, int QC, int PC>
__device__ __forceinline__ void tail_load(const PassArgs& A, long long base, int task, float2 (&r)[N1]) {
    const int P = PC ? PC : A.P;
    const int Q = QC ? QC : A.TP * P;
    const unsigned long long stepB = (unsigned long long)N2 * (unsigned)A.stride_i * (unsigned)P * 8u;
    const int b = task / Q, q = task - b * Q;
    const int t = q / P, p = q - t * P;
    const long long gi = (base + (long long)t * A.stride_t + (long long)b * A.stride_i) * P + p;
    const float2* lp = (MODE == MODE_FIRST ? A.psi : A.acc) + gi;
#pragma unroll
    for (int a = 0; a < N1; ++a) r[a] = ldg64(lp, stepB * a);
}

template <int N1, int N2, int MODE, int E, int QC, int PC, int NTC, int MINB>
__global__ void __launch_bounds__(NTC ? NTC : 320, MINB) pass_kernel(const __grid_constant__ PassArgs A) {
    extern __shared__ __align__(128) float2 smem[];
    constexpr int n = N1 * N2;
    constexpr bool TMA = QC != 0;                               // specialised kernels: tile by TMA bulk copies
    constexpr bool STACKED = TMA && MODE == MODE_FIRST;         // x pass
    using G = Geo<N1, N2, QC, PC, STACKED>;
    const int P = PC ? PC : A.P;
    const int Q = QC ? QC : A.TP * P;
    float2* tile = smem;
    float* sig = reinterpret_cast<float*>(tile + (TMA ? (size_t)G::tile_elems : (size_t)n * Q));
    __shared__ __align__(8) unsigned long long bar[N2];
    constexpr int NBAR = STACKED ? 1 : N2;
    constexpr bool FUSED = TMA && (32 % (QC ? QC : 7) == 0) && (NTC % 32 == 0);   // a warp owns whole rows of the tile
    // couple first: rows of one residue are owned by a warp, or by one full round of the CTA's task loop
    constexpr bool CF = FUSED || (TMA && NTC % (QC ? QC : 7) == 0 && (QC * N2) % (NTC ? NTC : 1) == 0);
    const int tid = threadIdx.x, nt = NTC ? NTC : blockDim.x;
    const int group = blockIdx.x / A.tiles_per_group, tin = blockIdx.x - group * A.tiles_per_group;
    const int valid = min(A.TP, A.pencils_per_group - tin * A.TP);
    const long long base = group * A.group_stride + (long long)tin * A.TP * A.stride_t;
    if constexpr (TMA) {
        if (tid < NBAR) {
            mbar_init(&bar[tid], 1);
            mbar_arrive_expect_tx(&bar[tid], (unsigned)(n / NBAR) * QC * 8u);
        }
        __syncthreads();
        tile_tma_load<N1, N2, QC, PC, STACKED>(A, tile, base, bar, tid, nt);
    }
    if (MODE == MODE_FIRST) build_sig<N1, N2>(A, sig, base, valid, tid, nt);
    phase_fwd1<N1, N2, E, QC, PC, STACKED, TMA, CF>(A, tile, base, valid, tid, nt, bar);
    __syncthreads();
    phase_mid<N1, N2, QC, PC, STACKED>(A, tile, tid, nt);
    const long long pencil0 = (long long)blockIdx.x * A.TP;
    if constexpr (CF) {
        // the first tail task's global loads are issued BEFORE the barrier, so they fly while the slower warps finish
        // phase 2 (the loads depend on nothing in shared memory; valid == TP in the specialised kernels)
        float2 r[N1];
        tail_load<N1, N2, MODE, QC, PC>(A, base, tid, r);
        __syncthreads();
        tail_task<N1, N2, MODE, E, QC, PC, STACKED, FUSED, CF>(A, tile, sig, base, valid, tid, pencil0, r, true);
#pragma unroll 1
        for (int task = tid + nt; task < Q * N2; task += nt) {
            float2 r2[N1];
            tail_task<N1, N2, MODE, E, QC, PC, STACKED, FUSED, CF>(A, tile, sig, base, valid, task, pencil0, r2, false);
        }
    } else {
        __syncthreads();
        if constexpr (!FUSED) {
            phase_inv1<N1, N2, QC, PC, STACKED>(A, tile, tid, nt);
            __syncthreads();
        }
#pragma unroll 1
        for (int task = tid; task < Q * N2; task += nt) {
            float2 r[N1];
            tail_task<N1, N2, MODE, E, QC, PC, STACKED, FUSED, CF>(A, tile, sig, base, valid, task, pencil0, r, false);
        }
    }
}
#endif

}  // namespace rtepass
