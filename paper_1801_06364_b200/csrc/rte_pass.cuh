// rte_pass.cuh — the per-axis pencil kernel of the P_N pseudospectral RTE step (sm_100a).
//
// One launch handles one axis a of the step (PAPER.md:123-127 re-designed).  The state is double
// buffered: every pass READS psi^n and ACCUMULATES into the buffer that becomes psi^{n+1} (eq.(11)):
//        FIRST (x axis)  new  = psi (1 - c dt sigma_l) + c dt q - c dt T_x   (scattering diagonal eq.(9), PML eq.(12),
//                                                                            source; plain stores)
//        ACC (other axes) new += -c dt T_a
// with  -c dt T_c = D_a ( sum_c' w^a_{cc'} psi_c' )  the streaming coupling (sparse l+-1, m, m+-1; eq.(6)/(10),
// PAPER.md:73-78) and D_a = IDFT (i k_a) DFT the spectral derivative along the axis (eq.(7)-(8),(10)).
// Specialised kernels (the BASELINE configurations; compile-time geometry):
//   0. the psi tile (TP adjacent pencils, all pairs of every cell) arrives in shared memory by TMA bulk copies
//   1. gather + couple the <= E source pairs of every column, first factor of DFT_n (N1-point), in place
//   2. twiddle, second factor (N2-point), multiply by i k_a (Nyquist zeroed), inverse second factor, conjugate twiddle
//   3. inverse first factor in registers, then
//      ACC:   ONE fire-and-forget vector reduction per element into the new buffer (red.global.add.v2.f32, SASS
//             REDG.ADD.F32x2, performed by the L2 at full HBM rate): the SM never waits for the accumulator, and since
//             every address receives exactly one reduction per pass the result does not depend on scheduling;
//      FIRST: psi is read again (L2 hit), combined with the Euler diagonal and the source, and stored.
// Generic kernels (any supported extent / order): registers -> DFT -> shared, phases 2, 3, coupling from the
// differentiated pencil, accumulator by load / add / store.
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

// MODE_RT (generic kernels): FIRST or ACC decided at run time by PassArgs::first, one instance per pencil length
enum { MODE_ACC = 0, MODE_FIRST = 1, MODE_RT = 2 };

struct PassArgs {
    // fields
    const float2* psi;      // [G][P]  state at t_n (input of the transform)
    float2* acc;            // [G][P]  accumulator: becomes the state at t_{n+1} after the last pass
    // tables (twiddles and wrapped integer wavenumbers live in constant memory, see c_tw / c_kw)
    const CplEntry* cpl;    // [P][kMaxE], unused entries: src = own pair, weights 0
    // diagonal + source (FIRST)
    const float* sa;        // [G] mu_a in Omega, mu_b in the PML
    const float* ss;        // [G] mu_s in Omega, 0 in the PML
    const float* gm;        // [G] g
    const int* deg;         // [2P] degree l of every slot
    float cdt;              // c * dt  (-1 when the kernels apply the steady-state operator L = T + sigma_l, rte_apply_operator)
    float ident;            // the Euler diagonal is  s_l = ident - cdt sigma_l : 1 for a time step, 0 for the operator
    int expo;               // generic kernels only: exponential (integrating-factor) Euler step, s_l = exp(-cdt sigma_l)
                            // multiplies psi AND the streaming term, the source carries phi_1 (rte_step_exp)
    int first;              // MODE_RT kernels: 1 = FIRST, 0 = ACC
    int first_axis;         // axis of the FIRST pass (0 = x, 2 = z): how the source box maps onto its pencils
    const float2* base;     // optional (FIRST pass): the store becomes  new = (scaled Euler update) + beta * base  — a Runge-Kutta
    float beta;             // stage combination fused into the pass (the scaling itself is in the tables: rte_lib.cu euler_update)
    const int* halt;        // optional device flag: non-zero => the launch does nothing (Krylov solver, converged early)
    const float2* tw;       // generic kernels: forward twiddles exp(-2 pi i j / n) of this axis, n entries (global)
    int nsig;               // N + 1 degrees
    float g_uniform;        // > 0: g is this number in every cell AND the kernel instance is a uniform-g one (UG): the
                            // diagonal table then holds 2 numbers per cell (build_sig); 0: N+1 numbers per cell
    const float* srcS;      // [ext z][ext y][ext x], already zero outside Omega
    const float* srcw;      // [2P] angular weight per slot
    int src_org[3], src_ext[3];
    float src_amp;          // c dt f(t_n); 0 => no source this step
    const float* src_amp_dev;   // optional: device location of c dt f(t_n) (CUDA-graph replay), read when src_amp != 0
    // geometry of this pass (cells)
    int stride_i;           // cell stride along the pencil
    int stride_t;           // cell stride between neighbouring pencils of a tile
    long long group_stride; // cell stride between pencil groups
    int pencils_per_group, tiles_per_group;
    int P, TP;
    int nx, ny;
};

// Pencil lengths of the SPECIALISED kernels and where their tables start in the constant arrays (the generic kernels
// take any even n = 2^a 3^b: twiddles from PassArgs::tw, wavenumbers by integer arithmetic).
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

// fire-and-forget  *p += v  on both halves (performed at the L2; flushes subnormals to zero, which is far below the
// parity tolerance).  One reduction per address per pass: deterministic.
__device__ __forceinline__ void red_add64(float2* p, unsigned long long byte_offset, float2 v) {
    asm volatile("red.global.add.v2.f32 [%0], {%1,%2};" ::"l"(reinterpret_cast<char*>(p) + byte_offset), "f"(v.x), "f"(v.y) : "memory");
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

// L2 prefetch of a contiguous global range (no destination in shared memory, nothing to wait for)
__device__ __forceinline__ void tma_prefetch_l2(const void* gmem_src, unsigned bytes) {
    asm volatile("cp.async.bulk.prefetch.L2.global [%0], %1;" ::"l"(gmem_src), "r"(bytes) : "memory");
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
    // One-pencil stacked tiles whose rows are not a multiple of 16 elements (P_5: 18 pairs): the phase-2 tasks of a half-warp
    // straddle two k1 blocks, N2 rows = N2*P elements apart — a multiple of 16 banks, i.e. a 2-way conflict.  A gap of PADB
    // elements after every block of N2 rows shifts consecutive blocks by 2 banks (ncu, cfg3 x pass: 20 % of the shared
    // wavefronts were conflicts).  SA = element stride between the rows i and i + N2.
    // (the interleaved y / z tiles of such records, rows of Q = 36 elements, have the same conflicts; padding them was measured
    // and changes nothing: those passes are HBM-bound)
    static constexpr int PADB = (STACKED && TPC == 1 && PC % 16 != 0 && (N2 * PC) % 16 == 0) ? 2 : 0;
    static constexpr int SA = N2 * SI + PADB;                // 0 when run-time (SI = 0, PADB = 0)
    static constexpr int ST = STACKED ? n * PC + pad + N1 * PADB : PC;
    static constexpr int tile_elems = STACKED ? TPC * ST : n * QC;
};

// ---- phase 0 (specialised kernels): the whole psi tile by TMA bulk copies ------------------------------------------------
template <int N1, int N2, int QC, int PC, bool STACKED>
__device__ __forceinline__ void tile_tma_load(const PassArgs& A, float2* tile, long long base, unsigned long long* bar, int tid,
                                              int nt) {
    using G = Geo<N1, N2, QC, PC, STACKED>;
    if (STACKED && G::PADB != 0) {
        // one pencil, one copy per block of N2 rows (N2*P*8 contiguous bytes) into its padded place
        constexpr unsigned blk_bytes = (unsigned)N2 * PC * 8u;
        for (int a = tid; a < N1; a += nt)
            tma_load_1d(tile + a * G::SA, reinterpret_cast<const char*>(A.psi + base * PC) + (size_t)a * blk_bytes, blk_bytes, bar);
    } else if (STACKED) {
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

// ---- source term along one pencil of the FIRST pass: c dt f(t_n) w_c S(r) for the cells inside the source box -------------
// ax = 0: x pencils (pencil = y + ny z, the position along the pencil is x); ax = 2: z pencils (pencil = x + nx y,
// position z).  (The y axis never carries the FIRST pass.)
struct SourceRow {
    bool on = false;
    float sw0 = 0.f, sw1 = 0.f;
    const float* S = nullptr;      // S at the box origin along this pencil
    int i0 = 0, ext = 0, stride = 1;
    // p = pair
    __device__ __forceinline__ SourceRow(const PassArgs& A, int ax, long long pencil, int p) {
        if (A.src_amp == 0.f) return;
        if (ax == 0) {
            const int by = (int)(pencil % A.ny) - A.src_org[1], bz = (int)(pencil / A.ny) - A.src_org[2];
            if (by < 0 || by >= A.src_ext[1] || bz < 0 || bz >= A.src_ext[2]) return;
            S = A.srcS + ((size_t)bz * A.src_ext[1] + by) * A.src_ext[0];
            i0 = A.src_org[0]; ext = A.src_ext[0]; stride = 1;
        } else {
            const int bx = (int)(pencil % A.nx) - A.src_org[0], by = (int)(pencil / A.nx) - A.src_org[1];
            if (bx < 0 || bx >= A.src_ext[0] || by < 0 || by >= A.src_ext[1]) return;
            S = A.srcS + (size_t)by * A.src_ext[0] + bx;
            i0 = A.src_org[2]; ext = A.src_ext[2]; stride = A.src_ext[0] * A.src_ext[1];
        }
        on = true;
        const float amp = A.src_amp_dev ? __ldg(A.src_amp_dev) : A.src_amp;
        sw0 = __ldg(A.srcw + 2 * p) * amp; sw1 = __ldg(A.srcw + 2 * p + 1) * amp;
    }
    __device__ __forceinline__ void add(int i, float2& e) const {
        if (!on) return;
        const int bi = i - i0;
        if (bi >= 0 && bi < ext) {
            const float v = __ldg(S + (size_t)bi * stride);
            e.x = fmaf(sw0, v, e.x); e.y = fmaf(sw1, v, e.y);
        }
    }
};

// ---- phase 1: first factor forward.  Generic: HBM -> registers -> DFT -> shared.  TMA: in place in shared ------------------
// CF ("couple first", specialised kernels): the streaming coupling is applied HERE, to the transform's input —
//   -c dt T_c = D_a ( sum_c' w^a_{cc'} psi_c' )      (constant weights commute with D_a; R18)
// so a column gathers its <= E source pairs from the freshly loaded tile, and the tail needs no neighbour data at all:
// one shared-memory store and E loads per element become E loads, and the tail runs without any barrier.  The
// gather reads rows that other columns of the same rows overwrite, hence the fence between gather and store: the rows
// of one residue b are owned by one warp (32 % Q == 0) or by one round of the whole CTA (nt % Q == 0).
template <int N1, int N2, int AX, int E, int QC, int PC, bool STACKED, bool TMA, bool CF>
__device__ __forceinline__ void phase_fwd1(const PassArgs& A, float2* tile, const float* sig, long long base, int valid,
                                           int tid, int nt, unsigned long long* bar) {
    using G = Geo<N1, N2, QC, PC, STACKED>;
    const int P = PC ? PC : A.P;
    const int Q = QC ? QC : A.TP * P;
    const int SI = G::SI ? G::SI : Q;
    const int ST = G::ST ? G::ST : P;
    const int SA = G::SA ? G::SA : N2 * SI;                  // stride between the rows i and i + N2
    const unsigned long long stepB = (unsigned long long)N2 * (unsigned)A.stride_i * (unsigned)P * 8u;
#pragma unroll 1
    for (int task = tid; task < Q * N2; task += nt) {
        const int b = task / Q, q = task - b * Q;
        const int t = q / P, p = q - t * P;
        float2* col = tile + b * SI + t * ST + p;
        float2 v[N1];
        if (CF) {
            // The specialised kernels are launched with E = 4 on the x and y axes and E = 2 on the z axis; the pair
            // layout guarantees 2 pure slots on x (diagonal blocks) and y (off-diagonal blocks) — rte_tables.h
            // PairLayout::npure, checked by the host before it picks these kernels.
            constexpr int NPURE = (E == 4) ? 2 : 0;
            constexpr bool PURE_DIAG = AX == 0;
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
                    const float2 d = srow[e][a * SA];
                    // slots [0, NPURE) hold purely diagonal (x pass) / purely off-diagonal (y pass) blocks: one packed FMA
                    if (e >= NPURE || PURE_DIAG) u = rtefft::cfma_diag(wd[e].x, wd[e].y, d, u);
                    if (e >= NPURE || !PURE_DIAG) u = rtefft::cfma_swap(ws[e].x, ws[e].y, d, u);
                }
                v[a] = u;
            }
            if (QC && 32 % (QC ? QC : 1) == 0) __syncwarp();
            else __syncthreads();
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
        for (int k1 = 0; k1 < N1; ++k1) col[k1 * SA] = v[k1];
    }
}

// ---- phase 2: twiddle, second factor forward, i k / n, second factor inverse, conjugate twiddle -----------------------
// LOWREG (instances that run 3+ CTAs per SM): the twiddles are fetched again for the conjugate multiply instead of
// being kept in N2 register pairs across the two transforms (constant-cache reads, off the load/store data path).
template <int N1, int N2, int QC, int PC, bool STACKED, bool LOWREG = false>
__device__ __forceinline__ void phase_mid(const PassArgs& A, float2* tile, int tid, int nt) {
    using G = Geo<N1, N2, QC, PC, STACKED>;
    constexpr int n = N1 * N2;
    constexpr bool CT = QC != 0;                      // specialised kernels: constant-memory tables
    constexpr int off = CT ? table_offset(n) : 0;
    const int P = PC ? PC : A.P;
    const int Q = QC ? QC : A.TP * P;
    const int SI = G::SI ? G::SI : Q;
#pragma unroll 1
    for (int task = tid; task < Q * N1; task += nt) {
        const int k1 = task / Q, q = task - k1 * Q;
        float2* row = tile + k1 * (G::SA ? G::SA : N2 * SI) + col_offset<G, STACKED>(q, P);
        float2 v[N2], w[N2];
#pragma unroll
        for (int b = 0; b < N2; ++b) v[b] = row[b * SI];
        int ti = 0;     // running twiddle index k1*b; LOWREG pins it so that the N2 indices are not precomputed and spilled
#pragma unroll
        for (int b = 1; b < N2; ++b) {
            ti += k1;
            if (LOWREG) asm volatile("" : "+r"(ti));
            w[b] = CT ? c_tw[off + ti] : __ldg(A.tw + ti);
            v[b] = rtefft::cmul(v[b], w[b]);
        }
        rtefft::dft_fwd<N2>(v);
#pragma unroll
        for (int k2 = 0; k2 < N2; ++k2) {
            // * i * wrapped(k), k = k1 + N1 k2: k below n/2, 0 at the Nyquist bin (R5), k - n above; 2 pi/(n dx)/n is in
            // the weights
            const int k = k1 + N1 * k2;
            const float kw = CT ? c_kw[off + k] : (float)(2 * k < n ? k : (2 * k == n ? 0 : k - n));
            v[k2] = rtefft::cscale(make_float2(-v[k2].y, v[k2].x), kw);
        }
        rtefft::dft_inv<N2>(v);
        ti = 0;
#pragma unroll
        for (int b = 1; b < N2; ++b) {
            ti += k1;
            if (LOWREG) asm volatile("" : "+r"(ti));
            const float2 wc = LOWREG ? (CT ? c_tw[off + ti] : __ldg(A.tw + ti)) : w[b];
            v[b] = rtefft::cmulc(v[b], wc);
        }
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

// Pitches of the per-tile diagonal table sig[l*sig_pitch_l + t*sig_pitch_t + i] (floats).  A reading warp spans degrees l,
// (with several pencils per tile) pencils t and, when a tile row is not a multiple of 32 columns, two neighbouring cells
// i: with the pencil pitch = 2 and the degree pitch = 4 (mod 32 banks) the lanes' banks 4 l + 2 t + {0, 1} are distinct for up
// to 8 degrees and 2 pencils (every BASELINE configuration); other shapes stay correct and may conflict.
#ifdef __CUDACC__
__host__ __device__
#endif
constexpr int sig_pitch_t(int n) { return n + 2; }
#ifdef __CUDACC__
__host__ __device__
#endif
constexpr int sig_pitch_l(int n, int TP) { return TP * (n + 2) + (36 - (TP * (n + 2)) % 32) % 32; }

// ---- FIRST only: per-tile table of the Euler diagonal  s_l(r) = 1 - c dt sigma_l(r) -----------------------------------
// sigma_l = mu_a + mu_s (1 - g^l) in Omega (eq.(9); g^l by repeated multiplication, R16),
//         = mu_b for every l in the PML, where the maps hold (mu_b, 0, g) (eq.(12)).
// Layout sig[l*sig_pitch_l + t*sig_pitch_t + i]: conflict-free to build (lanes = cells) and to read (lanes = degrees, pencils).
// (General form s_l = ident - c dt sigma_l: ident = 1 for a time step; ident = 0, c dt = -1 gives s_l = sigma_l, the
// diagonal of the steady-state operator L = T + sigma_l; expo: s_l = exp(-c dt sigma_l), generic kernels only.)
// Uniform g (A.g_uniform > 0): s_l = 1 - c dt (sa + ss (1 - g^l)) = A + B g^l with A = 1 - c dt (sa + ss), B = c dt ss,
// so the table holds the float2 (A, B) per cell and every thread keeps g^l of its two slots in registers: one
// broadcast 8-byte read per element instead of two 4-byte reads, and a quarter of the table-building work.
// The map values of the (at most MAXC) cells a thread is responsible for; loaded BEFORE the TMA issue loop so that their DRAM
// latency overlaps it (ncu: the first use of these loads was the kernel's hottest stall).
template <int MAXC>
struct SigCells { float sa[MAXC], ss[MAXC], g[MAXC]; };

template <int N1, int N2, int MAXC, int AX>
__device__ __forceinline__ void load_sig_cells(const PassArgs& A, SigCells<MAXC>& c, long long base, int valid, int tid, int nt) {
    constexpr int n = N1 * N2;
    const int ncell = n * A.TP;
#pragma unroll
    for (int k = 0; k < MAXC; ++k) {
        const int j = tid + k * nt;
        c.sa[k] = c.ss[k] = c.g[k] = 0.f;
        if (j < ncell) {
            const int t = j / n, i = j - t * n;
            if (t < valid) {
                // x pass: the tile's cells are contiguous (cell stride 1, pencil stride n)
                const long long cell = AX == 0 ? base + j : base + (long long)t * A.stride_t + (long long)i * A.stride_i;
                c.sa[k] = __ldg(A.sa + cell); c.ss[k] = __ldg(A.ss + cell);
                if (!(A.g_uniform > 0.f)) c.g[k] = __ldg(A.gm + cell);
            }
        }
    }
}

template <int N1, int N2, int MAXC>
__device__ __forceinline__ void build_sig(const PassArgs& A, float* sig, const SigCells<MAXC>& c, int tid, int nt) {
    constexpr int n = N1 * N2;
    const int ncell = n * A.TP;
    const bool ug = A.g_uniform > 0.f;
    float2* ab = reinterpret_cast<float2*>(sig);
    const int pl = sig_pitch_l(n, A.TP);
#pragma unroll
    for (int k = 0; k < MAXC; ++k) {
        const int j = tid + k * nt;
        if (j >= ncell) break;
        const int t = j / n, i = j - t * n;
        const float sa = c.sa[k], ss = c.ss[k], g = c.g[k];
        if (ug) {
            // pitch n + 1 per pencil: the lanes of a warp read the entries of TP pencils at the same position, and n is a
            // multiple of the 16 eight-byte banks (ncu, cfg2 x pass: a 4-way conflict on every table read)
            ab[t * (n + 1) + i] = make_float2(A.ident - A.cdt * (sa + ss), A.cdt * ss);
            continue;
        }
        float pw = 1.f;
        float* dst = sig + t * sig_pitch_t(n) + i;
        for (int l = 0; l < A.nsig; ++l) {
            const float a = A.cdt * fmaf(ss, 1.f - pw, sa);          // c dt sigma_l
            *dst = A.expo ? expf(-a) : A.ident - a;                  // exponential step: exact decay over the step
            pw *= g;
            dst += pl;
        }
    }
}

// generic kernels (run-time tile size): load and build in one loop
template <int N1, int N2>
__device__ __forceinline__ void build_sig(const PassArgs& A, float* sig, long long base, int valid, int tid, int nt) {
    for (int j0 = 0; j0 < N1 * N2 * A.TP; j0 += nt) {
        SigCells<1> c;
        // (tid + j0: one cell per thread and round)
        const int n = N1 * N2, j = tid + j0;
        c.sa[0] = c.ss[0] = c.g[0] = 0.f;
        if (j < n * A.TP) {
            const int t = j / n, i = j - t * n;
            if (t < valid) {
                const long long cell = base + (long long)t * A.stride_t + (long long)i * A.stride_i;
                c.sa[0] = __ldg(A.sa + cell); c.ss[0] = __ldg(A.ss + cell);
                if (!(A.g_uniform > 0.f)) c.g[0] = __ldg(A.gm + cell);
            }
        }
        build_sig<N1, N2, 1>(A, sig, c, tid + j0, nt);
    }
}

// ---- tail, specialised kernels: inverse first factor in registers, then one store / vector reduction per element ---------
// (the coupling was applied in phase 1; every thread owns its column, so there is no barrier and no neighbour data)
// FIRST: r holds the column's own psi (loaded by tail_load, the first task's before the phase-2 barrier).
template <int N1, int N2, int QC, int PC, int AX, bool BASE = false>
__device__ __forceinline__ void tail_load(const PassArgs& A, const float* sig, long long base, int task, float2 (&r)[N1]);

// LATE (FIRST instances whose register budget cannot hold the psi column next to the transform's): the re-read is issued
// after the inverse DFT instead of before it; the higher occupancy of those instances hides its latency.
template <int N1, int N2, int MODE, int QC, int PC, bool STACKED, bool UG, int AX, bool LATE = false, bool BASE = false>
__device__ __forceinline__ void tail_spec(const PassArgs& A, const float2* tile, const float* sig, long long base, int task,
                                          long long pencil0, float2 (&r)[N1]) {
    using G = Geo<N1, N2, QC, PC, STACKED>;
    constexpr int n = N1 * N2;
    constexpr int P = PC, Q = QC, SI = G::SI, ST = G::ST;
    const unsigned long long stepB = (unsigned long long)N2 * (unsigned)A.stride_i * (unsigned)P * 8u;
    const int b = task / Q, q = task - b * Q;
    const int t = q / P, p = q - t * P;
    const float2* col = tile + b * SI + t * ST + p;
    float2 v[N1];
#pragma unroll
    for (int k1 = 0; k1 < N1; ++k1) v[k1] = col[k1 * G::SA];
    if (MODE == MODE_FIRST) rtefft::dft_inv_swap<N1>(v);      // register pressure: see rte_fft.cuh
    else rtefft::dft_inv<N1>(v);
    if (MODE == MODE_FIRST && LATE) tail_load<N1, N2, QC, PC, AX, BASE>(A, sig, base, task, r);
    // x pass (AX == 0): the pencil is contiguous (cell stride 1, pencil stride n), so every address of the column is the
    // base plus a compile-time offset and folds into the instruction's immediate field
    float2* sp = AX == 0 ? A.acc + (base + (long long)t * n + b) * P + p
                         : A.acc + (base + (long long)t * A.stride_t + (long long)b * A.stride_i) * P + p;
    auto store = [&](int a, float2 e) {
        if (AX == 0) sp[a * (N2 * P)] = e;
        else stg64(sp, stepB * a, e);
    };
    if (MODE == MODE_FIRST) {
        constexpr int pl = sig_pitch_l(n, QC / PC), pt = sig_pitch_t(n);
        const int i0 = __ldg(A.deg + 2 * p) * pl + t * pt + b, i1 = __ldg(A.deg + 2 * p + 1) * pl + t * pt + b;
        const SourceRow src(A, AX, pencil0 + t, p);
        // (the source test is hoisted out of the element loops: almost every pencil lies outside the source box)
        if (BASE) {                 // r already holds s_l psi + beta base (tail_load)
#pragma unroll
            for (int a = 0; a < N1; ++a) {
                float2 e = rtefft::cadd(r[a], v[a]);
                src.add(a * N2 + b, e);
                store(a, e);
            }
        } else if (UG) {
            const float2* ab = reinterpret_cast<const float2*>(sig) + t * (n + 1) + b;
            float g0 = 1.f, g1 = 1.f;
            for (int l = __ldg(A.deg + 2 * p); l > 0; --l) g0 *= A.g_uniform;          // g^l by repeated multiplication (R16)
            for (int l = __ldg(A.deg + 2 * p + 1); l > 0; --l) g1 *= A.g_uniform;
            if (src.on) {
#pragma unroll
                for (int a = 0; a < N1; ++a) {
                    const float2 c = ab[a * N2];
                    float2 e = rtefft::cfma_diag(fmaf(c.y, g0, c.x), fmaf(c.y, g1, c.x), r[a], v[a]);
                    src.add(a * N2 + b, e);
                    store(a, e);
                }
            } else {
#pragma unroll
                for (int a = 0; a < N1; ++a) {
                    const float2 c = ab[a * N2];
                    store(a, rtefft::cfma_diag(fmaf(c.y, g0, c.x), fmaf(c.y, g1, c.x), r[a], v[a]));
                }
            }
        } else if (src.on) {
#pragma unroll
            for (int a = 0; a < N1; ++a) {
                float2 e = rtefft::cfma_diag(sig[i0 + a * N2], sig[i1 + a * N2], r[a], v[a]);
                src.add(a * N2 + b, e);
                store(a, e);
            }
        } else {
#pragma unroll
            for (int a = 0; a < N1; ++a) store(a, rtefft::cfma_diag(sig[i0 + a * N2], sig[i1 + a * N2], r[a], v[a]));
        }
    } else {
        // one running pointer instead of N1 precomputed 64-bit addresses (they would not fit the 3-CTA register budget)
        unsigned long long off = 0;
#pragma unroll
        for (int a = 0; a < N1; ++a) {
            red_add64(sp, off, v[a]);
            asm volatile("add.u64 %0, %0, %1;" : "+l"(off) : "l"(stepB));
        }
    }
}

// the psi re-read of one FIRST tail task, issued as early as possible
// BASE (x pass with a fused Runge-Kutta combination): the base field is loaded here too and folded in at once,
//   r = s_l psi + beta base   (s_l from the diagonal table, complete since the barrier after phase 1),
// so that both streams are in flight before the phase-2 barrier and the tail only adds the streaming term.
template <int N1, int N2, int QC, int PC, int AX, bool BASE>
__device__ __forceinline__ void tail_load(const PassArgs& A, const float* sig, long long base, int task, float2 (&r)[N1]) {
    constexpr int P = PC, Q = QC;
    const int b = task / Q, q = task - b * Q;
    const int t = q / P, p = q - t * P;
    if (AX == 0) {          // x pass: compile-time offsets (see tail_spec)
        const long long off = (base + (long long)t * (N1 * N2) + b) * P + p;
        const float2* lp = A.psi + off;
#pragma unroll
        for (int a = 0; a < N1; ++a) r[a] = lp[a * (N2 * P)];
        if (BASE) {
            constexpr int n = N1 * N2;
            constexpr int pl = sig_pitch_l(n, QC / PC), pt = sig_pitch_t(n);
            const int i0 = __ldg(A.deg + 2 * p) * pl + t * pt + b, i1 = __ldg(A.deg + 2 * p + 1) * pl + t * pt + b;
            const float2* xp = A.base + off;
            float2 x[N1];
#pragma unroll
            for (int a = 0; a < N1; ++a) x[a] = xp[a * (N2 * P)];
#pragma unroll
            for (int a = 0; a < N1; ++a)
                r[a] = make_float2(fmaf(sig[i0 + a * N2], r[a].x, A.beta * x[a].x), fmaf(sig[i1 + a * N2], r[a].y, A.beta * x[a].y));
        }
    } else {
        const unsigned long long stepB = (unsigned long long)N2 * (unsigned)A.stride_i * (unsigned)P * 8u;
        const float2* lp = A.psi + (base + (long long)t * A.stride_t + (long long)b * A.stride_i) * P + p;
#pragma unroll
        for (int a = 0; a < N1; ++a) r[a] = ldg64(lp, stepB * a);
    }
}

// ---- tail, generic kernels: coupling from the differentiated pencil + accumulate / integrate -----------------------------
// Exponential step (A.expo; rte_step_exp):  FIRST  new = s (psi + T_x) + phi_1 c dt q,   ACC  new += s T_a,
// s = exp(-c dt sigma_l) from the table, phi_1 = (1 - s)/(c dt sigma_l) = (1 - s)/(-ln s)  (1 where s = 1).
template <int N1, int N2, int E>
__device__ __forceinline__ void tail_generic(const PassArgs& A, const float2* tile, const float* sig, long long base, int valid,
                                             int task, long long pencil0, bool first) {
    constexpr int n = N1 * N2;
    const int P = A.P;
    const int Q = A.TP * P;
    const unsigned long long stepB = (unsigned long long)N2 * (unsigned)A.stride_i * (unsigned)P * 8u;
    const int b = task / Q, q = task - b * Q;
    const int t = q / P, p = q - t * P;
    if (t >= valid) return;
    // this pair's coupling list (unused entries point at the pair itself with zero weights)
    const float2* srow[E];
    float2 wd[E], ws[E];
#pragma unroll
    for (int e = 0; e < E; ++e) {
        const CplEntry* ce = A.cpl + p * kMaxE + e;
        srow[e] = tile + b * Q + t * P + __ldg(&ce->src);
        wd[e] = __ldg(reinterpret_cast<const float2*>(&ce->wd0));
        ws[e] = __ldg(reinterpret_cast<const float2*>(&ce->ws0));
    }
    const long long gi = (base + (long long)t * A.stride_t + (long long)b * A.stride_i) * P + p;
    float2* sp = A.acc + gi;
    float2 r[N1];
    // FIRST re-reads psi; the accumulating passes add their term by a fire-and-forget vector reduction like the
    // specialised kernels (one reduction per address per pass: deterministic), so they load nothing here
    if (first) {
#pragma unroll
        for (int a = 0; a < N1; ++a) r[a] = ldg64(A.psi + gi, stepB * a);
    }
    const float* s0 = sig;
    const float* s1 = sig;
    const bool table = first || A.expo;
    if (table) {
        const int pl = sig_pitch_l(n, A.TP), pt = sig_pitch_t(n);
        s0 = sig + __ldg(A.deg + 2 * p) * pl + t * pt + b;
        s1 = sig + __ldg(A.deg + 2 * p + 1) * pl + t * pt + b;
    }
    const SourceRow src(A, A.first_axis, pencil0 + t, p);
#pragma unroll
    for (int a = 0; a < N1; ++a) {
        float2 T = make_float2(0.f, 0.f);
#pragma unroll
        for (int e = 0; e < E; ++e) {
            const float2 d = srow[e][(a * N2) * Q];
            T = rtefft::cfma_diag(wd[e].x, wd[e].y, d, T);
            T = rtefft::cfma_swap(ws[e].x, ws[e].y, d, T);
        }
        if (A.expo) {
            const float e0 = s0[a * N2], e1 = s1[a * N2];
            if (first) {
                r[a] = make_float2(e0 * (r[a].x + T.x), e1 * (r[a].y + T.y));
                float2 qv = make_float2(0.f, 0.f);
                src.add(a * N2 + b, qv);
                if (qv.x != 0.f) r[a].x = fmaf(e0 < 1.f ? (1.f - e0) / -logf(e0) : 1.f, qv.x, r[a].x);
                if (qv.y != 0.f) r[a].y = fmaf(e1 < 1.f ? (1.f - e1) / -logf(e1) : 1.f, qv.y, r[a].y);
            } else {
                r[a] = make_float2(e0 * T.x, e1 * T.y);
            }
        } else if (first) {
            r[a] = rtefft::cfma_diag(s0[a * N2], s1[a * N2], r[a], T);
            src.add(a * N2 + b, r[a]);
        } else {
            r[a] = T;
        }
    }
    if (first) {
        if (A.base != nullptr) {          // Runge-Kutta stage combination fused into the store
            const float2* bp = A.base + gi;
#pragma unroll
            for (int a = 0; a < N1; ++a) {
                const float2 x = ldg64(bp, stepB * a);
                r[a].x = fmaf(A.beta, x.x, r[a].x); r[a].y = fmaf(A.beta, x.y, r[a].y);
            }
        }
#pragma unroll
        for (int a = 0; a < N1; ++a) stg64(sp, stepB * a, r[a]);
    } else {
#pragma unroll
        for (int a = 0; a < N1; ++a) red_add64(sp, stepB * a, r[a]);
    }
}

// Largest block of a generic instance: small register transforms leave room for more threads (a tile of many
// coefficients allows one CTA per SM only, so the block is the occupancy), 32/36-point ones need their 255 registers.
#ifdef __CUDACC__
__host__ __device__
#endif
constexpr int generic_max_threads(int N1, int N2) {
    return (N1 > 32 || N2 > 32) ? 224 : ((N1 > 24 || N2 > 24) ? 256 : ((N1 > 18 || N2 > 18) ? 320 : ((N1 > 9 || N2 > 12) ? 512 : 640)));
}

// UG (specialised FIRST kernels only): uniform g, the 2-number diagonal table (build_sig); the host picks the instance.
// AX (specialised kernels): the axis of the pass — x tiles of several pencils use the stacked layout, x / y have pure
// coupling slots, the FIRST pass maps the source box onto its pencils by AX.
template <int N1, int N2, int MODE, int E, int QC, int PC, int NTC, int MINB, bool UG = false, int AX = 0, bool BASE = false>
__global__ void __launch_bounds__(NTC ? NTC : generic_max_threads(N1, N2), MINB) pass_kernel(const __grid_constant__ PassArgs A) {
    extern __shared__ __align__(128) float2 smem[];
    constexpr int n = N1 * N2;
    constexpr bool TMA = QC != 0;                                             // specialised kernels: tile by TMA bulk copies
    // x pass: pencils are contiguous in memory -> the tile is filled by a few large bulk copies ("stacked" layout; with
    // one pencil per tile it coincides with the interleaved one).  ncu: the 384 per-row copies of the one-pencil x tile
    // cost 8 % of the kernel's stall samples in their lane-serialised issue loop.
    constexpr bool STACKED = TMA && AX == 0;
    using G = Geo<N1, N2, QC, PC, STACKED>;
    // couple first needs the rows of one residue owned by a warp (32 % Q == 0) or by one full round of the CTA's task
    // loop (nt % Q == 0, whole rounds); all specialised configurations qualify (checked here at compile time)
    constexpr bool CF = TMA;
    static_assert(!TMA || ((32 % (QC ? QC : 1) == 0 && NTC % 32 == 0) ||
                           (NTC % (QC ? QC : 1) == 0 && (QC * N2) % (NTC ? NTC : 1) == 0)),
                  "specialised geometry must let a warp or a CTA round own whole tile rows");
    // the first tail task runs unguarded (task = tid < Q*N2) and the __syncwarp branch of phase 1 needs whole warps
    static_assert(!TMA || (QC * N2 >= NTC && (QC * N2) % 32 == 0), "specialised geometry: Q*N2 >= block size, whole warps");
    static_assert(MODE != MODE_RT || !TMA, "run-time FIRST/ACC is for the generic kernels");
    if (A.halt != nullptr && *reinterpret_cast<const volatile int*>(A.halt) != 0) return;   // uniform: whole grid
    const bool first = MODE == MODE_RT ? A.first != 0 : MODE == MODE_FIRST;
    const int P = PC ? PC : A.P;
    const int Q = QC ? QC : A.TP * P;
    float2* tile = smem;
    float* sig = reinterpret_cast<float*>(tile + (TMA ? (size_t)G::tile_elems : (size_t)n * Q));
    __shared__ __align__(8) unsigned long long bar[N2];
    constexpr int NBAR = STACKED ? 1 : N2;
    const int tid = threadIdx.x, nt = NTC ? NTC : blockDim.x;
    // specialised kernels: whole tiles only (the host checks pencils % TP == 0); their x pass has one group of contiguous pencils
    constexpr int TPC = QC / (PC ? PC : 1);
    const int group = (TMA && AX == 0) ? 0 : blockIdx.x / A.tiles_per_group, tin = blockIdx.x - group * A.tiles_per_group;
    const int valid = TMA ? TPC : min(A.TP, A.pencils_per_group - tin * A.TP);
    const long long base = (TMA && AX == 0) ? (long long)blockIdx.x * (TPC * n)
                                            : group * A.group_stride + (long long)tin * A.TP * A.stride_t;
    const long long pencil0 = (long long)blockIdx.x * A.TP;
    if constexpr (TMA) {
        constexpr int MAXC = (n * (QC / (PC ? PC : 1)) + (NTC ? NTC : 1) - 1) / (NTC ? NTC : 1);
        SigCells<MAXC> cells;
        if (MODE == MODE_FIRST) load_sig_cells<N1, N2, MAXC, AX>(A, cells, base, valid, tid, nt);   // in flight during the TMA issue
        if (tid < NBAR) {
            mbar_init(&bar[tid], 1);
            mbar_arrive_expect_tx(&bar[tid], (unsigned)(n / NBAR) * QC * 8u);
        }
        __syncthreads();
        tile_tma_load<N1, N2, QC, PC, STACKED>(A, tile, base, bar, tid, nt);
        if constexpr (BASE && AX == 0) {
            // the Runge-Kutta base field of this (contiguous) x tile is read in the tail: bring it into L2 now, so that those
            // loads cost an L2 hit like the psi re-read instead of a DRAM round trip each
            constexpr unsigned tile_bytes = (unsigned)n * QC * 8u;
            constexpr unsigned piece = tile_bytes % 16384u == 0 ? 16384u : (tile_bytes % 4096u == 0 ? 4096u : tile_bytes);
            for (unsigned j = tid; j < tile_bytes / piece; j += nt)
                tma_prefetch_l2(reinterpret_cast<const char*>(A.base + base * PC) + (size_t)j * piece, piece);
        }
        if (MODE == MODE_FIRST) build_sig<N1, N2, MAXC>(A, sig, cells, tid, nt);                 // read in the tail, two barriers later
    } else {
        if (first || A.expo) build_sig<N1, N2>(A, sig, base, valid, tid, nt);
    }
    phase_fwd1<N1, N2, AX, E, QC, PC, STACKED, TMA, CF>(A, tile, sig, base, valid, tid, nt, bar);
    __syncthreads();
    phase_mid<N1, N2, QC, PC, STACKED, (MINB >= 3 && N2 >= 16)>(A, tile, tid, nt);
    if constexpr (CF) {
        float2 r[N1];
        // FIRST: the first tail task's psi re-read is issued BEFORE the barrier and flies while the slower warps finish
        // phase 2 (the loads depend on nothing in shared memory)
        constexpr bool LATE = MODE == MODE_FIRST && 65536 / ((NTC ? NTC : 1) * MINB) < 80;
        if (MODE == MODE_FIRST && !LATE) tail_load<N1, N2, QC, PC, AX, BASE>(A, sig, base, tid, r);
        __syncthreads();
        tail_spec<N1, N2, MODE, QC, PC, STACKED, UG, AX, LATE, BASE>(A, tile, sig, base, tid, pencil0, r);
#pragma unroll 1
        for (int task = tid + nt; task < Q * N2; task += nt) {
            float2 r2[N1];
            if (MODE == MODE_FIRST && !LATE) tail_load<N1, N2, QC, PC, AX, BASE>(A, sig, base, task, r2);
            tail_spec<N1, N2, MODE, QC, PC, STACKED, UG, AX, LATE, BASE>(A, tile, sig, base, task, pencil0, r2);
        }
    } else {
        __syncthreads();
        phase_inv1<N1, N2, QC, PC, STACKED>(A, tile, tid, nt);
        __syncthreads();
#pragma unroll 1
        for (int task = tid; task < Q * N2; task += nt) tail_generic<N1, N2, E>(A, tile, sig, base, valid, task, pencil0, first);
    }
}
#endif

}  // namespace rtepass
