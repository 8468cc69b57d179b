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
//   3-D: the m = 0 fields a_l^0 (l = 0..N) come first, two per pair, even with even and odd with odd degree (a zero
//        pad field completes the last pair when N+1 is odd); then one pair (a_l^m, b_l^m) for every m >= 1, l >= m.  This makes every pair with m >= 1 the
//        paper's complex coefficient psi_l^m up to a factor, so x/y/z coupling maps pairs to pairs.
//   2-D: (a_0, pad), then (a_m, b_m), m = 1..N.
// Slot 0 is always coefficient 0 (the fluence).
#pragma once
#include <cmath>
#include <complex>
#include <cstdint>
#include <limits>
#include <map>
#include <mutex>
#include <utility>
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

// base slot order (before the bank-conflict permutation of pair positions, see PairLayout below):
// ext_of_slot[s] = external coefficient index (or -1 for the pad), deg_of_slot[s] = l (2-D: m)
inline void base_slot_order(int dim, int N, std::vector<int>& ext_of_slot, std::vector<int>& deg_of_slot) {
    ext_of_slot.clear(); deg_of_slot.clear();
    if (dim == 3) {
        // m = 0 fields: even degrees paired among themselves, odd degrees among themselves (a_0,a_2), (a_4,a_6), ...,
        // (a_1,a_3), ...; a left-over even and a left-over odd degree share a pair, a single left-over gets the pad.
        // The z coupling links l to l+-1, i.e. even to odd, so a pair then has at most 2 source pairs on the z axis
        // (3 with (a_l, a_l+1) pairs, which couple to themselves) and the z kernels gather 2 entries instead of 3.
        std::vector<int> ev, od, rest;
        for (int l = 0; l <= N; ++l) (l % 2 ? od : ev).push_back(l);
        auto emit = [&](std::vector<int>& v) {
            size_t k = 0;
            for (; k + 1 < v.size(); k += 2)
                for (int h = 0; h < 2; ++h) { ext_of_slot.push_back(ia3(v[k + h], 0)); deg_of_slot.push_back(v[k + h]); }
            if (k < v.size()) rest.push_back(v[k]);
        };
        emit(ev); emit(od);
        for (int l : rest) { ext_of_slot.push_back(ia3(l, 0)); deg_of_slot.push_back(l); }
        if (rest.size() % 2) { ext_of_slot.push_back(-1); deg_of_slot.push_back(0); }
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
inline void pair_coupling_of(int dim, int N, int axis, const std::vector<int>& ext,
                             std::vector<std::vector<PairEntry>>& out) {
    std::vector<double> A[3];
    coupling_real(dim, N, A);
    const int C = num_coeffs(dim, N);
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

// ---- pair layout: positions of the pairs inside a cell record, and the entry order of the coupling lists ----------------
// The specialised pass kernels gather, per coupling entry e, one 8-byte element per lane from the shared-memory tile:
// lane (row i, pencil t, position pp) reads tile[i*Q + t*P + pos(src_e(pair at pp))] (x pass with several pencils per
// tile: pencils stacked with pitch = P mod 16 (mod 16)).  A 64-bit shared load is served half-warp by half-warp; two
// lanes of a half-warp that hit the same 8-byte bank (address mod 16) at different addresses cost an extra wavefront.
// Both the position of every pair in the record and the order of a pair's entries are free, so they are chosen here to
// minimise those extra wavefronts (deterministic simulated annealing; the pair that holds coefficient 0 stays at
// position 0 because the fluence read-out takes slot 0).  Pure layout: no arithmetic of the method depends on it.
struct PairLayout {
    int P = 0;
    std::vector<int> pos;                          // pos[base pair] = position in the record
    std::vector<int> inv;                          // inv[position] = base pair
    std::vector<std::vector<int>> slots[3];        // slots[axis][position][e] = source POSITION, or -1 (unused)
    int cost0 = 0, cost = 0, ideal = 0;            // modelled wavefronts: base layout, chosen layout, conflict-free
    // slots [0, npure[axis]) of EVERY pair hold entries whose 2x2 block is purely diagonal (x, z axes) / purely
    // off-diagonal (y axis) or empty, so the kernels spend one packed FMA per element on them instead of two
    int npure[3] = {0, 0, 0};
};

inline int layout_tp(int dim, int N) {   // pencils per tile assumed by the model (the specialised kernels' choice)
    const int P = (dim == 3 ? ((N + 1) + ((N + 1) % 2)) / 2 + N * (N + 1) / 2 : N + 1);
    int tp = 1;
    while (tp * P < 32 && tp < 8) tp *= 2;
    return tp;
}

// pencils per x tile assumed by the model (= the specialised kernels' choice, rte_lib.cu kSpec TPx).  The 18-pair records
// of P_5 use ONE pencil per x tile: a contiguous tile whose own-element accesses are conflict-free (two stacked pencils
// conflict at half of the row boundaries) and small enough for 3 CTAs per SM (measured: x pass -6 %; at 2 CTAs per SM
// the same tile was 14 % slower).
inline int layout_tp_x(int dim, int N) { return (dim == 3 && N == 5) ? 1 : layout_tp(dim, N); }

// modelled wavefronts of ONE axis' gathers for a candidate layout
inline int layout_cost_axis(int P, int TP, int axis, int E, const std::vector<int>& pos, const std::vector<int>& inv,
                            const std::vector<std::vector<int>>& src /* [base pair][e] base pair or -1 */) {
    const int Q = TP * P;
    int g = 32, h = Q;
    while (h) { const int r = g % h; g = h; h = r; }
    const int period = 32 * Q / g;                 // tasks after which the warp/row alignment repeats
    const bool stacked = axis == 0 && TP > 1;
    int tot = 0;
    for (int w0 = 0; w0 < period; w0 += 16) {      // one half-warp at a time
        int abase[16], pr[16];
        for (int lane = 0; lane < 16; ++lane) {
            const int task = w0 + lane, b = task / Q, q = task - b * Q, t = q / P;
            pr[lane] = inv[q - t * P];
            abase[lane] = stacked ? t * (P % 16) + b * P + 4096 * t : b * Q + t * P;
        }
        for (int e = 0; e < E; ++e) {
            int worst = 1, cnt[16] = {0}, seen[16][16];
            for (int lane = 0; lane < 16; ++lane) {
                int s = src[pr[lane]][e];
                if (s < 0) s = pr[lane];
                const int addr = abase[lane] + pos[s], bank = addr & 15;
                bool dup = false;
                for (int k = 0; k < cnt[bank]; ++k) if (seen[bank][k] == addr) dup = true;
                if (!dup) { seen[bank][cnt[bank]++] = addr; if (cnt[bank] > worst) worst = cnt[bank]; }
            }
            tot += worst;
        }
    }
    return tot;
}

inline const PairLayout& pair_layout(int dim, int N) {
    static std::mutex mu;
    static std::map<std::pair<int, int>, PairLayout> cache;
    std::lock_guard<std::mutex> lock(mu);
    auto it = cache.find({dim, N});
    if (it != cache.end()) return it->second;
    PairLayout L;
    std::vector<int> ext, deg;
    base_slot_order(dim, N, ext, deg);
    const int P = (int)ext.size() / 2, naxes = dim, TP = layout_tp(dim, N);
    L.P = P;
    // coupling structure in base pair indices, padded with -1 to E entries per axis
    int E[3] = {4, 4, 4};
    std::vector<std::vector<int>> src[3], pure[3];
    for (int a = 0; a < naxes; ++a) {
        std::vector<std::vector<PairEntry>> pe;
        pair_coupling_of(dim, N, a, ext, pe);
        size_t mx = 0;
        for (auto& v : pe) mx = v.size() > mx ? v.size() : mx;
        if (dim == 3 && a == 2 && mx <= 2) E[a] = 2;            // the z kernels read 2 entries (rte_lib.cu launch_spec)
        if ((int)mx > E[a]) E[a] = (int)mx;
        // entries of the axis' pure kind (block diagonal on x and z, off-diagonal on y) go first; gaps count as pure
        src[a].assign(P, {});
        pure[a].assign(P, {});
        int np = E[a];
        for (int p = 0; p < P; ++p) {
            std::vector<int> first, rest;
            for (auto& en : pe[p]) {
                const bool diag_only = en.w01 == 0.f && en.w10 == 0.f, swap_only = en.w00 == 0.f && en.w11 == 0.f;
                ((a == 1 ? swap_only : diag_only) ? first : rest).push_back(en.src);
            }
            const int npair = E[a] - (int)rest.size();          // pure entries + gaps of this pair
            if (npair < np) np = npair;
            for (int s : first) { src[a][p].push_back(s); pure[a][p].push_back(1); }
            while ((int)src[a][p].size() + (int)rest.size() < E[a]) { src[a][p].push_back(-1); pure[a][p].push_back(1); }
            for (int s : rest) { src[a][p].push_back(s); pure[a][p].push_back(0); }
        }
        L.npure[a] = np < 0 ? 0 : np;
    }
    std::vector<int> pos(P), inv(P);
    for (int p = 0; p < P; ++p) pos[p] = inv[p] = p;
    int cax[3] = {0, 0, 0};
    const int TPX = layout_tp_x(dim, N);
    auto tp_of = [&](int a) { return a == 0 ? TPX : TP; };
    for (int a = 0; a < naxes; ++a) cax[a] = layout_cost_axis(P, tp_of(a), a, E[a], pos, inv, src[a]);
    L.cost0 = cax[0] + cax[1] + cax[2];
    {
        L.ideal = 0;
        for (int a = 0; a < naxes; ++a) {
            int g = 32, h = tp_of(a) * P;
            while (h) { const int r = g % h; g = h; h = r; }
            L.ideal += E[a] * (32 * tp_of(a) * P / g) / 16;
        }
    }
    // deterministic annealing: swap two pair positions (never position 0) or permute one pair's entry order
    uint64_t rng = 0x9E3779B97F4A7C15ull ^ ((uint64_t)dim << 32) ^ (uint64_t)N;
    auto next = [&]() { rng = rng * 6364136223846793005ull + 1442695040888963407ull; return (uint32_t)(rng >> 33); };
    int cur = L.cost0, best = cur;
    std::vector<int> best_pos = pos;
    std::vector<std::vector<int>> best_src[3] = {src[0], src[1], src[2]};
    double T = 2.0;
    // larger records: base layout (generic kernels).  The 18-pair records of P_5 (configs[3]) get a ten times longer,
    // slower schedule (3 s, once per process): it reaches a conflict-free x axis and 1.06 / 1.11 of ideal on y / z.
    const bool slow = dim == 3 && N == 5;
    const int iters = (P > 2 && P <= 40 && cur > L.ideal) ? (slow ? 200000 : 20000) : 0;
    const double cool = slow ? 0.99995 : 0.9995;
    for (int itn = 0; itn < iters && best > L.ideal; ++itn) {
        const bool swap_move = (next() & 1) && P > 2;
        int i = 0, j = 0, a = 0, p = 0, oldpure_swap[2] = {0, 0};
        std::vector<int> old;
        if (swap_move) {
            i = 1 + (int)(next() % (uint32_t)(P - 1));
            j = 1 + (int)(next() % (uint32_t)(P - 1));
            if (i == j) continue;
            std::swap(pos[i], pos[j]);
            inv[pos[i]] = i; inv[pos[j]] = j;
        } else {
            a = (int)(next() % (uint32_t)naxes); p = (int)(next() % (uint32_t)P);
            old = src[a][p];
            // swap two slots of this pair; an entry may enter the pure class [0, npure) only if it is pure
            const int e1 = (int)(next() % (uint32_t)E[a]), e2 = (int)(next() % (uint32_t)E[a]);
            const int lo = e1 < e2 ? e1 : e2, hi = e1 < e2 ? e2 : e1;
            if (lo == hi || (lo < L.npure[a] && !pure[a][p][hi])) continue;
            std::swap(src[a][p][lo], src[a][p][hi]);
            std::swap(pure[a][p][lo], pure[a][p][hi]);
            oldpure_swap[0] = lo; oldpure_swap[1] = hi;
        }
        int nax[3] = {cax[0], cax[1], cax[2]};
        for (int k = 0; k < naxes; ++k)
            if (swap_move || k == a) nax[k] = layout_cost_axis(P, tp_of(k), k, E[k], pos, inv, src[k]);
        const int c = nax[0] + nax[1] + nax[2];
        const double u = (double)(next() & 0xFFFFFF) / 16777216.0;
        if (c <= cur || u < std::exp((double)(cur - c) / T)) { cur = c; for (int k = 0; k < 3; ++k) cax[k] = nax[k]; }
        else if (swap_move) { std::swap(pos[i], pos[j]); inv[pos[i]] = i; inv[pos[j]] = j; }
        else { src[a][p] = old; std::swap(pure[a][p][oldpure_swap[0]], pure[a][p][oldpure_swap[1]]); }
        T = T * cool > 0.05 ? T * cool : 0.05;
        if (cur < best) { best = cur; best_pos = pos; for (int k = 0; k < 3; ++k) best_src[k] = src[k]; }
    }
    L.cost = best;
    L.pos = best_pos;
    L.inv.assign(P, 0);
    for (int p = 0; p < P; ++p) L.inv[L.pos[p]] = p;
    for (int a = 0; a < naxes; ++a) {
        L.slots[a].assign(P, {});
        for (int pp = 0; pp < P; ++pp)
            for (int s : best_src[a][L.inv[pp]]) L.slots[a][pp].push_back(s < 0 ? -1 : L.pos[s]);
    }
    return cache.emplace(std::make_pair(dim, N), std::move(L)).first->second;
}

// internal slot order = base order with the pairs moved to their layout positions
inline void slot_order(int dim, int N, std::vector<int>& ext_of_slot, std::vector<int>& deg_of_slot) {
    std::vector<int> ext, deg;
    base_slot_order(dim, N, ext, deg);
    const PairLayout& L = pair_layout(dim, N);
    ext_of_slot.assign(ext.size(), -1); deg_of_slot.assign(deg.size(), 0);
    for (int p = 0; p < L.P; ++p)
        for (int h = 0; h < 2; ++h) {
            ext_of_slot[2 * L.pos[p] + h] = ext[2 * p + h];
            deg_of_slot[2 * L.pos[p] + h] = deg[2 * p + h];
        }
}

// coupling by pair POSITION, entries in the layout's order (gaps, src = -1, carry zero weights)
inline void pair_coupling(int dim, int N, int axis, std::vector<std::vector<PairEntry>>& out) {
    std::vector<int> ext, deg;
    slot_order(dim, N, ext, deg);
    std::vector<std::vector<PairEntry>> pe;
    pair_coupling_of(dim, N, axis, ext, pe);
    const PairLayout& L = pair_layout(dim, N);
    out.assign(L.P, {});
    for (int pp = 0; pp < L.P; ++pp)
        for (int s : L.slots[axis][pp]) {
            PairEntry en{-1, 0.f, 0.f, 0.f, 0.f};
            if (s >= 0)
                for (auto& c : pe[pp]) if (c.src == s) en = c;
            out[pp].push_back(en);
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

// Supported pencil lengths: every EVEN n = 2^a 3^b in [16, 1024] (odd lengths have no Nyquist bin and are not offered:
// reading R5 is stated for even n), with the N1 x N2 split of the two-factor transform (N1-point transforms in role I,
// N2-point in role II; both are register DFTs of rte_fft.cuh, radix 2/3/4).  X(N1, N2) for the generic kernels'
// dispatch (rte_lib.cu): one kernel instance per row.
#define RTE_SPLITS(X)                                                                                                  \
    X(4, 4) X(6, 3) X(6, 4) X(4, 8) X(6, 6) X(4, 12) X(9, 6) X(8, 8) X(9, 8) X(8, 12) X(12, 9) X(8, 16) X(12, 12)      \
    X(18, 9) X(12, 16) X(18, 12) X(16, 16) X(18, 16) X(18, 18) X(24, 16) X(24, 18) X(27, 18) X(32, 16) X(24, 24)       \
    X(27, 24) X(32, 24) X(32, 27) X(36, 27) X(32, 32)
inline bool split_of(int n, int& N1, int& N2) {
#define RTE_SPLIT_CASE(A, B) if (n == (A) * (B)) { N1 = (A); N2 = (B); return true; }
    RTE_SPLITS(RTE_SPLIT_CASE)
#undef RTE_SPLIT_CASE
    return false;
}

// ---- forward-Euler stability bound (R10; "time-steps of the order of 100 fs provide stability") ---
// Eigenvalues of a small dense complex matrix: elementary reduction to Hessenberg form, then shifted QR with deflation
// (Wilkinson shift, an exceptional shift every 10 sweeps).  a is n x n row-major and is destroyed.
inline bool eig_complex(std::vector<std::complex<double>>& a, int n, std::vector<std::complex<double>>& lam) {
    typedef std::complex<double> cd;
    auto H = [&](int i, int j) -> cd& { return a[(size_t)i * n + j]; };
    for (int m = 1; m < n - 1; ++m) {                        // Gaussian similarity transforms with pivoting
        int piv = m;
        for (int i = m + 1; i < n; ++i) if (std::abs(H(i, m - 1)) > std::abs(H(piv, m - 1))) piv = i;
        if (std::abs(H(piv, m - 1)) == 0.0) continue;
        if (piv != m) {
            for (int j = 0; j < n; ++j) std::swap(H(piv, j), H(m, j));
            for (int i = 0; i < n; ++i) std::swap(H(i, piv), H(i, m));
        }
        for (int i = m + 1; i < n; ++i) {
            const cd f = H(i, m - 1) / H(m, m - 1);
            if (f == cd(0, 0)) continue;
            for (int j = 0; j < n; ++j) H(i, j) -= f * H(m, j);
            for (int k = 0; k < n; ++k) H(k, m) += f * H(k, i);
        }
    }
    lam.assign(n, cd(0, 0));
    int hi = n - 1, iter = 0;
    double scale = 0;
    for (auto& v : a) scale = std::max(scale, std::abs(v));
    if (scale == 0.0) return true;
    while (hi >= 0) {
        int l = hi;
        while (l > 0) {
            const double sd = std::abs(H(l - 1, l - 1)) + std::abs(H(l, l));
            if (std::abs(H(l, l - 1)) <= 1e-15 * (sd > 0 ? sd : scale)) break;
            --l;
        }
        if (l == hi) { lam[hi] = H(hi, hi); --hi; iter = 0; continue; }
        if (++iter > 400) return false;
        cd mu;
        if (iter % 10 == 0) mu = H(hi, hi) + cd(std::abs(H(hi, hi - 1)), 0.0);
        else {                                              // eigenvalue of the trailing 2x2 closest to H(hi,hi)
            const cd p = H(hi - 1, hi - 1), q = H(hi - 1, hi), r = H(hi, hi - 1), t = H(hi, hi);
            const cd tr = p + t, det = p * t - q * r, disc = std::sqrt(tr * tr * 0.25 - det);
            const cd e1 = tr * 0.5 + disc, e2 = tr * 0.5 - disc;
            mu = std::abs(e1 - t) < std::abs(e2 - t) ? e1 : e2;
        }
        for (int i = l; i <= hi; ++i) H(i, i) -= mu;
        std::vector<cd> cs(hi - l), sn(hi - l);
        for (int k = l; k < hi; ++k) {                      // R = G_{hi-1} ... G_l (H - mu)
            const cd x = H(k, k), y = H(k + 1, k);
            const double r = std::sqrt(std::norm(x) + std::norm(y));
            const cd c = r > 0 ? x / r : cd(1, 0), s2 = r > 0 ? y / r : cd(0, 0);
            cs[k - l] = c; sn[k - l] = s2;
            for (int j = k; j < n; ++j) {
                const cd u = H(k, j), v = H(k + 1, j);
                H(k, j) = std::conj(c) * u + std::conj(s2) * v;
                H(k + 1, j) = -s2 * u + c * v;
            }
        }
        for (int k = l; k < hi; ++k) {                      // R G_l^H ... G_{hi-1}^H
            const cd c = cs[k - l], s2 = sn[k - l];
            const int top = k + 2 <= hi ? k + 2 : hi;
            for (int i = 0; i <= top; ++i) {
                const cd u = H(i, k), v = H(i, k + 1);
                H(i, k) = u * c + v * s2;
                H(i, k + 1) = -u * std::conj(s2) + v * std::conj(c);
            }
        }
        for (int i = l; i <= hi; ++i) H(i, i) += mu;
    }
    return true;
}

// dt <= -2 Re(lambda)/|lambda|^2 over the eigenvalues of M(k) = -c (i k A_axis + diag sigma_l), sigma_l = mu_a + mu_s (1 - g^l),
// k along z (3-D) / x (2-D) — rotational invariance — on 200 magnitudes up to the corner Nyquist sqrt(d) (pi/dx)(1 - 2/n).
// A_axis only links coefficients of one azimuthal order, so M(k) is handled one connected block at a time.
inline bool stable_dt_bound(int dim, int N, int n, double dx, double c, double mu_a, double mu_s, double g, double& bound) {
    typedef std::complex<double> cd;
    const int C = num_coeffs(dim, N);
    if (C < 0 || n < 4 || !(dx > 0) || !(c > 0)) return false;
    std::vector<double> A[3];
    coupling_real(dim, N, A);
    const std::vector<double>& Az = A[dim == 3 ? 2 : 0];
    std::vector<int> ext, deg, degc(C, 0);
    base_slot_order(dim, N, ext, deg);
    for (size_t s = 0; s < ext.size(); ++s) if (ext[s] >= 0) degc[ext[s]] = deg[s];
    std::vector<double> sigma(C);
    for (int i = 0; i < C; ++i) sigma[i] = mu_a + mu_s * (1.0 - std::pow(g, (double)degc[i]));
    // connected components of the coupling graph
    std::vector<int> comp(C, -1);
    std::vector<std::vector<int>> blocks;
    for (int s0 = 0; s0 < C; ++s0) {
        if (comp[s0] >= 0) continue;
        std::vector<int> blk{s0};
        comp[s0] = (int)blocks.size();
        for (size_t h = 0; h < blk.size(); ++h)
            for (int j = 0; j < C; ++j)
                if (comp[j] < 0 && (Az[(size_t)blk[h] * C + j] != 0.0 || Az[(size_t)j * C + blk[h]] != 0.0)) {
                    comp[j] = comp[s0];
                    blk.push_back(j);
                }
        blocks.push_back(blk);
    }
    const double kmax = std::sqrt((double)dim) * 3.14159265358979323846 / dx * (1.0 - 2.0 / (double)n);
    bound = std::numeric_limits<double>::infinity();
    for (int ik = 1; ik <= 200; ++ik) {
        const double k = kmax * (double)ik / 200.0;
        for (const auto& blk : blocks) {
            const int m = (int)blk.size();
            std::vector<cd> M((size_t)m * m), lam;
            for (int i = 0; i < m; ++i)
                for (int j = 0; j < m; ++j)
                    M[(size_t)i * m + j] = -c * (cd(0.0, k * Az[(size_t)blk[i] * C + blk[j]]) + (i == j ? cd(sigma[blk[i]], 0.0) : cd(0, 0)));
            if (!eig_complex(M, m, lam)) return false;
            for (const cd& l : lam) {
                const double b2 = -2.0 * l.real() / std::norm(l);
                if (b2 < bound) bound = b2;
            }
        }
    }
    return true;
}

}  // namespace rtetab
