// rte_tables.h — host-side coefficient layer of the product library: real-basis streaming coupling, the internal
// "pair" ordering of coefficients, wavenumbers and twiddles.  Host C++ only (no device code, no oracle code).
//
// Coupling: written out directly in the REAL basis from eq.(6)/(10) with the 1/(2l+1) on all
// three brackets (R1) and the real harmonics of R6 — the explicit formulas of DESIGN.md R7 (3-D) and R8
// (2-D).  (The oracle derives its tables another way: complex eq.(10) + change of basis; tests compare both with
// quadrature.)
//
// Internal storage: the C real fields are regrouped into P = Cp/2 "pairs" so that one complex FFT differentiates two
// real fields at once (D_a is a real operator, so D(u + i v) = Du + i Dv):
//   3-D: the m = 0 fields a_l^0 (l = 0..N) come first, two per pair (a zero pad field completes the last pair when
//        N+1 is odd); then one pair (a_l^m, b_l^m) for every m >= 1, l >= m.  This makes every pair with m >= 1 the
//        paper's complex coefficient psi_l^m up to a factor, so x/y/z coupling maps pairs to pairs.
//   2-D: (a_0, pad), then (a_m, b_m), m = 1..N.
// Slot 0 is always coefficient 0 (the fluence).
#pragma once
#include <cmath>
#include <cstdint>
#include <vector>

namespace rtetab {

inline int num_coeffs(int dim, int N) {
    if (N < 1 || (dim != 2 && dim != 3)) return -1;
    return dim == 3 ? (N + 1) * (N + 1) : 2 * N + 1;
}

// external index of a_l^m (m>=0) / b_l^m (m>=1)
inline int ia3(int l, int m) { return l * l + l + m; }
inline int ib3(int l, int m) { return l * l + l - m; }

inline double alpha_lm(int l, int m) { int v = (l + m) * (l - m); return v > 0 ? std::sqrt((double)v) : 0.0; }
inline double beta_lm(int l, int m) { int v = (l + m) * (l + m - 1); return v > 0 ? std::sqrt((double)v) : 0.0; }

// A[axis][c*C + c'] : T_c = sum_c' A d_axis psi_c'
inline void coupling_real(int dim, int N, std::vector<double> A[3]) {
    const int C = num_coeffs(dim, N);
    for (int a = 0; a < 3; ++a) A[a].assign((size_t)C * C, 0.0);
    auto add = [&](int axis, int row, int col, double w) { A[axis][(size_t)row * C + col] += w; };
    if (dim == 3) {
        auto exists = [&](int l, int m) { return l >= 0 && l <= N && m >= 0 && m <= l; };
        const double rs2 = 1.0 / std::sqrt(2.0), s2 = std::sqrt(2.0);
        for (int l = 0; l <= N; ++l) {
            const double f = 1.0 / (2.0 * l + 1.0);
            for (int m = 0; m <= l; ++m) {
                const int ra = ia3(l, m), rb = ib3(l, m);
                // d/dz [ alpha_{l+1}^m X_{l+1}^m + alpha_l^m X_{l-1}^m ],  X = a or b
                if (exists(l + 1, m)) {
                    add(2, ra, ia3(l + 1, m), f * alpha_lm(l + 1, m));
                    if (m >= 1) add(2, rb, ib3(l + 1, m), f * alpha_lm(l + 1, m));
                }
                if (exists(l - 1, m)) {
                    add(2, ra, ia3(l - 1, m), f * alpha_lm(l, m));
                    if (m >= 1) add(2, rb, ib3(l - 1, m), f * alpha_lm(l, m));
                }
                if (m == 0) {
                    // T^a_{l0} = f/sqrt2 [ -beta_l^0 (dx a_{l-1}^1 + dy b_{l-1}^1) + beta_{l+1}^1 (dx a_{l+1}^1 + dy b_{l+1}^1) ]
                    if (exists(l - 1, 1)) {
                        const double w = -f * rs2 * beta_lm(l, 0);
                        add(0, ra, ia3(l - 1, 1), w); add(1, ra, ib3(l - 1, 1), w);
                    }
                    if (exists(l + 1, 1)) {
                        const double w = f * rs2 * beta_lm(l + 1, 1);
                        add(0, ra, ia3(l + 1, 1), w); add(1, ra, ib3(l + 1, 1), w);
                    }
                } else {
                    // neighbours with m-1 (A^0 = sqrt2 a^0, B^0 = 0 when m-1 = 0):
                    //   T^a += f/2 [ beta_l^m (dx A - dy B)_{l-1}^{m-1} - beta_{l+1}^{-m+1} (dx A - dy B)_{l+1}^{m-1} ]
                    //   T^b += f/2 [ beta_l^m (dy A + dx B)_{l-1}^{m-1} - beta_{l+1}^{-m+1} (dy A + dx B)_{l+1}^{m-1} ]
                    const double sc = (m - 1 == 0) ? s2 : 1.0;
                    const int lps[2] = {l - 1, l + 1};
                    const double lo[2] = {beta_lm(l, m), -beta_lm(l + 1, -m + 1)};
                    for (int j = 0; j < 2; ++j) {
                        if (!exists(lps[j], m - 1)) continue;
                        const double w = 0.5 * f * lo[j] * sc;
                        add(0, ra, ia3(lps[j], m - 1), w);
                        add(1, rb, ia3(lps[j], m - 1), w);
                        if (m - 1 >= 1) {
                            add(1, ra, ib3(lps[j], m - 1), -w);
                            add(0, rb, ib3(lps[j], m - 1), w);
                        }
                    }
                    // neighbours with m+1:
                    //   T^a += f/2 [ -beta_l^{-m} (dx a + dy b)_{l-1}^{m+1} + beta_{l+1}^{m+1} (dx a + dy b)_{l+1}^{m+1} ]
                    //   T^b += f/2 [ -beta_l^{-m} (dx b - dy a)_{l-1}^{m+1} + beta_{l+1}^{m+1} (dx b - dy a)_{l+1}^{m+1} ]
                    const double hi[2] = {-beta_lm(l, -m), beta_lm(l + 1, m + 1)};
                    for (int j = 0; j < 2; ++j) {
                        if (!exists(lps[j], m + 1)) continue;
                        const double w = 0.5 * f * hi[j];
                        add(0, ra, ia3(lps[j], m + 1), w);
                        add(1, ra, ib3(lps[j], m + 1), w);
                        add(0, rb, ib3(lps[j], m + 1), w);
                        add(1, rb, ia3(lps[j], m + 1), -w);
                    }
                }
            }
        }
    } else {
        // R8: T_0 = dx a_1 + dy b_1 ; m>=1: T^a_m = 1/2 (dx A_{m-1} - dy B_{m-1}) + 1/2 (dx a_{m+1} + dy b_{m+1}),
        //                                  T^b_m = 1/2 (dy A_{m-1} + dx B_{m-1}) + 1/2 (dx b_{m+1} - dy a_{m+1}),
        //     with (A_0, B_0) = (a_0, 0) and a_{N+1} = b_{N+1} = 0.   c=0 a_0; c=2m-1 a_m; c=2m b_m.
        auto ia = [](int m) { return m == 0 ? 0 : 2 * m - 1; };
        auto ib = [](int m) { return 2 * m; };
        if (N >= 1) { add(0, 0, ia(1), 1.0); add(1, 0, ib(1), 1.0); }
        for (int m = 1; m <= N; ++m) {
            add(0, ia(m), ia(m - 1), 0.5);
            add(1, ib(m), ia(m - 1), 0.5);
            if (m - 1 >= 1) { add(1, ia(m), ib(m - 1), -0.5); add(0, ib(m), ib(m - 1), 0.5); }
            if (m + 1 <= N) {
                add(0, ia(m), ia(m + 1), 0.5); add(1, ia(m), ib(m + 1), 0.5);
                add(0, ib(m), ib(m + 1), 0.5); add(1, ib(m), ia(m + 1), -0.5);
            }
        }
    }
}

// internal slot order: ext_of_slot[s] = external coefficient index (or -1 for the pad), deg_of_slot[s] = l (2-D: m)
inline void slot_order(int dim, int N, std::vector<int>& ext_of_slot, std::vector<int>& deg_of_slot) {
    ext_of_slot.clear(); deg_of_slot.clear();
    if (dim == 3) {
        for (int l = 0; l <= N; ++l) { ext_of_slot.push_back(ia3(l, 0)); deg_of_slot.push_back(l); }
        if ((N + 1) % 2) { ext_of_slot.push_back(-1); deg_of_slot.push_back(0); }
        for (int m = 1; m <= N; ++m)
            for (int l = m; l <= N; ++l) {
                ext_of_slot.push_back(ia3(l, m)); deg_of_slot.push_back(l);
                ext_of_slot.push_back(ib3(l, m)); deg_of_slot.push_back(l);
            }
    } else {
        ext_of_slot.push_back(0); deg_of_slot.push_back(0);
        ext_of_slot.push_back(-1); deg_of_slot.push_back(0);
        for (int m = 1; m <= N; ++m) {
            ext_of_slot.push_back(2 * m - 1); deg_of_slot.push_back(m);
            ext_of_slot.push_back(2 * m); deg_of_slot.push_back(m);
        }
    }
}

struct PairEntry { int src; float w00, w01, w10, w11; };   // out.x += w00 in.x + w01 in.y ; out.y += w10 in.x + w11 in.y

// coupling regrouped by pairs: for output pair po the list of (source pair, 2x2 block)
inline void pair_coupling(int dim, int N, int axis, std::vector<std::vector<PairEntry>>& out) {
    std::vector<double> A[3];
    coupling_real(dim, N, A);
    const int C = num_coeffs(dim, N);
    std::vector<int> ext, deg;
    slot_order(dim, N, ext, deg);
    const int P = (int)ext.size() / 2;
    out.assign(P, {});
    for (int po = 0; po < P; ++po)
        for (int ps = 0; ps < P; ++ps) {
            double w[2][2] = {{0, 0}, {0, 0}};
            bool any = false;
            for (int r = 0; r < 2; ++r)
                for (int c = 0; c < 2; ++c) {
                    const int er = ext[2 * po + r], ec = ext[2 * ps + c];
                    if (er < 0 || ec < 0) continue;
                    w[r][c] = A[axis][(size_t)er * C + ec];
                    if (w[r][c] != 0.0) any = true;
                }
            if (any) out[po].push_back({ps, (float)w[0][0], (float)w[0][1], (float)w[1][0], (float)w[1][1]});
        }
}

// wavenumbers with the Nyquist bin zeroed (R5), already divided by n (the inverse DFT normalisation)
inline void kappa_over_n(int n, double dx, std::vector<float>& k) {
    k.resize(n);
    const double two_pi = 6.283185307179586476925286766559;
    for (int j = 0; j < n; ++j) {
        int f = (2 * j < n) ? j : ((2 * j == n) ? 0 : j - n);
        k[j] = (float)(two_pi * (double)f / ((double)n * dx) / (double)n);
    }
}

// forward twiddles exp(-2 pi i j / n), j = 0..n-1, rounded once from fp64
inline void twiddles(int n, std::vector<float>& tw /* 2n: re, im */) {
    tw.resize(2 * (size_t)n);
    const double two_pi = 6.283185307179586476925286766559;
    for (int j = 0; j < n; ++j) {
        tw[2 * j] = (float)std::cos(two_pi * j / n);
        tw[2 * j + 1] = (float)(-std::sin(two_pi * j / n));
    }
}

// supported pencil lengths and their N1 x N2 split (N1-point transforms in role I, N2-point in role II)
inline bool split_of(int n, int& N1, int& N2) {
    switch (n) {
        case 16: N1 = 4; N2 = 4; return true;
        case 32: N1 = 4; N2 = 8; return true;
        case 48: N1 = 4; N2 = 12; return true;
        case 64: N1 = 8; N2 = 8; return true;
        case 96: N1 = 8; N2 = 12; return true;
        case 128: N1 = 8; N2 = 16; return true;
        case 192: N1 = 12; N2 = 16; return true;
        case 256: N1 = 16; N2 = 16; return true;
        case 384: N1 = 24; N2 = 16; return true;
        case 512: N1 = 32; N2 = 16; return true;
        default: return false;
    }
}

}  // namespace rtetab
