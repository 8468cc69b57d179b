// rte_oracle.cpp — fp64 CPU ORACLE for the pseudospectral P_N radiative-transport time step.
//
// THIS IS TEST INFRASTRUCTURE, NOT THE PRODUCT.  Only tests/, __graft_entry__.smoke() and the
// cpu_baseline / --impl reference legs of bench.py may load it.  It shares no code, header, table or
// constant generator with the CUDA path under paper_1801_06364_b200/csrc/, and neither includes the other.
//
// What it computes (all citations are PAPER.md line numbers of arXiv:1801.06364, Powell/Cox/Arridge):
//   * the P_N moment system, eq.(6), with alpha/beta of PAPER.md:78;
//   * the spatial Fourier transform eq.(7)-(8) PAPER.md:84-90, replaced by its discrete counterpart;
//   * the k-space streaming operator eq.(10) PAPER.md:98 and the ODE system eq.(9) PAPER.md:94;
//   * the forward-Euler step eq.(11) PAPER.md:104;
//   * the perfectly matched layer eq.(12) PAPER.md:113-119 with the half-cosine profile of PAPER.md:165.
// The paper's three-stage recipe is followed literally by formulation 0 ("literal"):
//   complex psi_l^m for all m in [-l,l]  ->  d-dimensional DFT of every field  ->  eq.(10) in k-space
//   ->  inverse DFT  ->  pointwise potential  ->  time step.
// Formulation 1 ("per-axis") is the same mathematics written as  T = sum_a A_a D_a psi  with the real-basis
// coupling matrices A_a obtained from the complex ones by the change of basis of DESIGN.md reading R6, and the
// 1-D spectral derivative D_a = IDFT_a( i k_a DFT_a(.) ); it exists so that big grids fit in memory and so that
// the two can be checked against each other (pin P12).
//
// Readings of the paper that this file takes:
//   R1  the 1/(2l+1) factor of eq.(10) multiplies all three brackets (eq.(6) as printed encloses only the first);
//   R2  forward transform with exp(-ik.r)  =>  d/dx_a -> +i k_a  (eq.(10) as printed carries the opposite sign);
//   R3  psi_{n+1} = psi_n - c dt ( T + sigma_l psi_n ) + c dt q_n  (eq.(11) as printed has the loss terms growing);
//   R4  "(mu_t mu_s g^l)" of PAPER.md:126 is mu_t - mu_s g^l;
//   R5  k_a[j] = 2 pi j/(n dx) (j<n/2), 0 (j=n/2), 2 pi (j-n)/(n dx) (j>n/2); inverse carries 1/n;
//   R6  real basis a_l^m (cos-type, m>=0), b_l^m (sin-type, m>=1):
//         psi_l^m = (-1)^m (a - i b)/sqrt2,  psi_l^{-m} = (a + i b)/sqrt2,  psi_l^0 = a_l^0   (m>0);
//   R8  2-D "circular harmonic" system: phi = (1/2pi) sum_m psi_m e^{i m theta}, psi_m = a_m - i b_m,
//         T_m = 1/2 (dx - i dy) psi_{m-1} + 1/2 (dx + i dy) psi_{m+1},  sigma_m = mu_a + mu_s (1 - g^|m|);
//   R9  fluence = coefficient 0;
//   R11 PML: depth p_a = max(W-i, i-(n-1-W), 0), delta = max_a p_a / W,
//         mu_b = mu_lo + (mu_hi-mu_lo) (1-cos(pi delta))/2 ; in the PML sigma_l = mu_b for every l, q = 0;
//   R14 the source is sampled at t_n.
//
// Parity pins for every function here live in tests/test_oracle_pins.py (P1..P16); none is "parity unpinned".
// Besides the paper's forward Euler there is one NON-PAPER integrator, SSP-RK3, built from the same
// Euler update; it is pinned by the stability polynomial of a single Fourier mode (P13).  SURVEY §8(f1)/(f2) add the
// steady-state operator L = T + sigma_l (P14), a plain restarted GMRES on it (P15: dense solve, closed form, true
// residual) and the exponential / integrating-factor Euler step (P16: exact uniform decay and source response).
//
// Coefficient order (external, = the C-ABI's):  3-D  c = l*l + l + m  (m>=0 -> a_l^m, m<0 -> b_l^|m|);
//                                                2-D  c = 0 -> a_0, c = 2m-1 -> a_m, c = 2m -> b_m.
// Field layout: [c][z][y][x], x fastest.
//
// Plain and slow on purpose: own recursive mixed-radix DFT, dense loops, OpenMP over pencils / cells only.

#include <cmath>
#include <complex>
#include <cstdint>
#include <cstdlib>
#include <cstring>
#include <vector>
#ifdef _OPENMP
#include <omp.h>
#endif

typedef std::complex<double> cd;
static const double PI = 3.14159265358979323846264338327950288;

// ------------------------------------------------------------------------------------------------------------
// Own DFT ("the continuous Fourier transform replaced with its discrete counterpart").
// X[k] = sum_j x[j] exp(sign * 2 pi i j k / n), sign = -1 forward (eq.(8)), +1 inverse (unnormalised).
// Recursive decimation in time on the smallest prime factor; any n.
// ------------------------------------------------------------------------------------------------------------
struct Dft {
    int n, sign;
    std::vector<cd> w;  // w[j] = exp(sign 2 pi i j / n), each by a direct cos/sin
    Dft(int n_, int sign_) : n(n_), sign(sign_), w(n_) {
        for (int j = 0; j < n; ++j) {
            double ang = sign * 2.0 * PI * (double)j / (double)n;
            w[j] = cd(std::cos(ang), std::sin(ang));
        }
    }
    static int spf(int m) {
        for (int p = 2; p * p <= m; ++p)
            if (m % p == 0) return p;
        return m;
    }
    // out[0..m) = DFT_m of in[0], in[is], in[2 is], ...; twiddle step in w is n/m
    void rec(const cd* in, long is, cd* out, int m) const {
        if (m == 1) { out[0] = in[0]; return; }
        const int p = spf(m), q = m / p, ws = n / m;
        for (int r = 0; r < p; ++r) rec(in + r * is, is * p, out + (long)r * q, q);
        std::vector<cd> t(p), u(p);
        for (int k = 0; k < q; ++k) {
            for (int r = 0; r < p; ++r) t[r] = out[(long)r * q + k];
            for (int s = 0; s < p; ++s) {
                cd acc(0, 0);
                const long kk = k + (long)q * s;
                for (int r = 0; r < p; ++r) acc += t[r] * w[((r * kk) % m) * ws];
                u[s] = acc;
            }
            for (int s = 0; s < p; ++s) out[k + (long)q * s] = u[s];
        }
    }
    void run(const cd* in, long is, cd* out) const { rec(in, is, out, n); }
};

// Wavenumbers, reading R5.
static void wavenumbers(int n, double dx, double* k) {
    for (int j = 0; j < n; ++j) {
        int f;
        if (2 * j < n) f = j;
        else if (2 * j == n) f = 0;
        else f = j - n;
        k[j] = 2.0 * PI * (double)f / ((double)n * dx);
    }
}

// ------------------------------------------------------------------------------------------------------------
// Coefficient bookkeeping
// ------------------------------------------------------------------------------------------------------------
static int num_coeffs(int dim, int N) { return dim == 3 ? (N + 1) * (N + 1) : 2 * N + 1; }
// complex index: 3-D (l,m) -> l*l+l+m ; 2-D m in [-N,N] -> m+N
static int cidx3(int l, int m) { return l * l + l + m; }

// alpha, beta of PAPER.md:78 (zero where the argument of the root is not positive)
static double alpha(int l, int m) { int v = (l + m) * (l - m); return v > 0 ? std::sqrt((double)v) : 0.0; }
static double beta(int l, int m) { int v = (l + m) * (l + m - 1); return v > 0 ? std::sqrt((double)v) : 0.0; }

// Complex-basis coupling of eq.(10) with R1: T_lm = sum_{l'm'} [ Ax dx + Ay dy + Az dz ] psi_l'm'.
// (dx - i dy) contributes  +1 to Ax and -i to Ay;  (dx + i dy) contributes +1 to Ax and +i to Ay.
static void coupling_complex3(int N, std::vector<cd>& Ax, std::vector<cd>& Ay, std::vector<cd>& Az) {
    const int C = (N + 1) * (N + 1);
    Ax.assign((size_t)C * C, cd(0, 0)); Ay = Ax; Az = Ax;
    auto present = [&](int l, int m) { return l >= 0 && l <= N && std::abs(m) <= l; };
    for (int l = 0; l <= N; ++l)
        for (int m = -l; m <= l; ++m) {
            const int r = cidx3(l, m);
            const double f = 1.0 / (2.0 * l + 1.0);
            // d/dz [ alpha_{l+1}^m psi_{l+1}^m + alpha_l^m psi_{l-1}^m ]
            if (present(l + 1, m)) Az[(size_t)r * C + cidx3(l + 1, m)] += f * alpha(l + 1, m);
            if (present(l - 1, m)) Az[(size_t)r * C + cidx3(l - 1, m)] += f * alpha(l, m);
            // -1/2 (dx - i dy) [ beta_l^m psi_{l-1}^{m-1} - beta_{l+1}^{-m+1} psi_{l+1}^{m-1} ]
            if (present(l - 1, m - 1)) {
                const double w = -0.5 * f * beta(l, m);
                Ax[(size_t)r * C + cidx3(l - 1, m - 1)] += w;
                Ay[(size_t)r * C + cidx3(l - 1, m - 1)] += w * cd(0, -1);
            }
            if (present(l + 1, m - 1)) {
                const double w = +0.5 * f * beta(l + 1, -m + 1);
                Ax[(size_t)r * C + cidx3(l + 1, m - 1)] += w;
                Ay[(size_t)r * C + cidx3(l + 1, m - 1)] += w * cd(0, -1);
            }
            // -1/2 (dx + i dy) [ -beta_l^{-m} psi_{l-1}^{m+1} + beta_{l+1}^{m+1} psi_{l+1}^{m+1} ]
            if (present(l - 1, m + 1)) {
                const double w = +0.5 * f * beta(l, -m);
                Ax[(size_t)r * C + cidx3(l - 1, m + 1)] += w;
                Ay[(size_t)r * C + cidx3(l - 1, m + 1)] += w * cd(0, +1);
            }
            if (present(l + 1, m + 1)) {
                const double w = -0.5 * f * beta(l + 1, m + 1);
                Ax[(size_t)r * C + cidx3(l + 1, m + 1)] += w;
                Ay[(size_t)r * C + cidx3(l + 1, m + 1)] += w * cd(0, +1);
            }
        }
}

// 2-D complex coupling (reading R8): T_m = 1/2 (dx - i dy) psi_{m-1} + 1/2 (dx + i dy) psi_{m+1}, |m|<=N.
static void coupling_complex2(int N, std::vector<cd>& Ax, std::vector<cd>& Ay) {
    const int C = 2 * N + 1;
    Ax.assign((size_t)C * C, cd(0, 0)); Ay = Ax;
    for (int m = -N; m <= N; ++m) {
        const int r = m + N;
        if (m - 1 >= -N) { Ax[(size_t)r * C + (m - 1 + N)] += 0.5; Ay[(size_t)r * C + (m - 1 + N)] += cd(0, -0.5); }
        if (m + 1 <= N)  { Ax[(size_t)r * C + (m + 1 + N)] += 0.5; Ay[(size_t)r * C + (m + 1 + N)] += cd(0, +0.5); }
    }
}

// Change of basis, reading R6 (3-D) / R8 (2-D):  psi_complex = U psi_real ;  psi_real = Uinv psi_complex.
static void basis_matrices(int dim, int N, std::vector<cd>& U, std::vector<cd>& Uinv) {
    const int C = num_coeffs(dim, N);
    U.assign((size_t)C * C, cd(0, 0)); Uinv = U;
    const double s = 1.0 / std::sqrt(2.0);
    if (dim == 3) {
        for (int l = 0; l <= N; ++l) {
            U[(size_t)cidx3(l, 0) * C + cidx3(l, 0)] = 1.0;
            Uinv[(size_t)cidx3(l, 0) * C + cidx3(l, 0)] = 1.0;
            for (int m = 1; m <= l; ++m) {
                const double sg = (m % 2) ? -1.0 : 1.0;
                const int ia = cidx3(l, m), ib = cidx3(l, -m);     // real: a_l^m at c(l,m), b_l^m at c(l,-m)
                const int ip = cidx3(l, m), im = cidx3(l, -m);     // complex: psi_l^m, psi_l^{-m}
                U[(size_t)ip * C + ia] = sg * s;  U[(size_t)ip * C + ib] = cd(0, -sg * s);
                U[(size_t)im * C + ia] = s;       U[(size_t)im * C + ib] = cd(0, s);
                // inverse = conjugate transpose (the 2x2 block is unitary)
                Uinv[(size_t)ia * C + ip] = sg * s;          Uinv[(size_t)ia * C + im] = s;
                Uinv[(size_t)ib * C + ip] = cd(0, sg * s);   Uinv[(size_t)ib * C + im] = cd(0, -s);
            }
        }
    } else {
        // real order: c=0 a_0; c=2m-1 a_m; c=2m b_m.  complex order: m+N.
        U[(size_t)N * C + 0] = 1.0; Uinv[(size_t)0 * C + N] = 1.0;
        for (int m = 1; m <= N; ++m) {
            const int ia = 2 * m - 1, ib = 2 * m, ip = N + m, im = N - m;
            U[(size_t)ip * C + ia] = 1.0; U[(size_t)ip * C + ib] = cd(0, -1);   // psi_m = a - i b
            U[(size_t)im * C + ia] = 1.0; U[(size_t)im * C + ib] = cd(0, +1);   // psi_{-m} = a + i b
            Uinv[(size_t)ia * C + ip] = 0.5;          Uinv[(size_t)ia * C + im] = 0.5;
            Uinv[(size_t)ib * C + ip] = cd(0, 0.5);   Uinv[(size_t)ib * C + im] = cd(0, -0.5);
        }
    }
}

static void matmul(const std::vector<cd>& A, const std::vector<cd>& B, std::vector<cd>& R, int C) {
    R.assign((size_t)C * C, cd(0, 0));
    for (int i = 0; i < C; ++i)
        for (int k = 0; k < C; ++k) {
            const cd a = A[(size_t)i * C + k];
            if (a == cd(0, 0)) continue;
            for (int j = 0; j < C; ++j) R[(size_t)i * C + j] += a * B[(size_t)k * C + j];
        }
}

// Real-basis coupling A^R_a = Uinv A^C_a U; returns the largest |imaginary part| (must be round-off).
static double coupling_real(int dim, int N, int axis, std::vector<double>& A) {
    const int C = num_coeffs(dim, N);
    std::vector<cd> Ax, Ay, Az, U, Ui, T, R;
    if (dim == 3) coupling_complex3(N, Ax, Ay, Az);
    else { coupling_complex2(N, Ax, Ay); Az.assign((size_t)C * C, cd(0, 0)); }
    basis_matrices(dim, N, U, Ui);
    const std::vector<cd>& Ac = axis == 0 ? Ax : (axis == 1 ? Ay : Az);
    matmul(Ac, U, T, C);
    matmul(Ui, T, R, C);
    A.resize((size_t)C * C);
    double im = 0;
    for (size_t i = 0; i < A.size(); ++i) { A[i] = R[i].real(); im = std::fmax(im, std::fabs(R[i].imag())); }
    return im;
}

// degree l of external coefficient c (2-D: |m|), used by the scattering diagonal
static void degrees(int dim, int N, std::vector<int>& L) {
    const int C = num_coeffs(dim, N);
    L.resize(C);
    if (dim == 3) { for (int l = 0; l <= N; ++l) for (int m = -l; m <= l; ++m) L[cidx3(l, m)] = l; }
    else { L[0] = 0; for (int m = 1; m <= N; ++m) { L[2 * m - 1] = m; L[2 * m] = m; } }
}

// ------------------------------------------------------------------------------------------------------------
// The solver
// ------------------------------------------------------------------------------------------------------------
struct Oracle {
    int dim, nx, ny, nz, N, C;
    long G;
    double dx, dt, c;
    std::vector<double> mu_a, mu_s, g;       // per cell (already expanded from scalars)
    std::vector<double> mu_b;                // PML attenuation per cell (0 in Omega)
    std::vector<unsigned char> inside;       // 1 in Omega
    std::vector<int> L;                      // degree per coefficient
    std::vector<double> psi, psi_new;        // [C][G]
    std::vector<double> A[3];                // real-basis coupling per axis
    std::vector<cd> Ac[3];                   // complex-basis coupling per axis
    std::vector<cd> U, Ui;
    // source: q_c(r,t) = w_c S(r) f(t)
    std::vector<double> src_w, src_S;
    int src_org[3], src_ext[3], src_kind;
    double src_t0, src_sigt;
    long step_count;
};

static void pml_map(int dim, int nx, int ny, int nz, int W, double mu_lo, double mu_hi, double* mu_b,
                    unsigned char* inside) {
    const int n[3] = {nx, ny, nz};
    for (int z = 0; z < nz; ++z)
        for (int y = 0; y < ny; ++y)
            for (int x = 0; x < nx; ++x) {
                const int i[3] = {x, y, z};
                int p = 0;
                for (int a = 0; a < dim; ++a) {
                    int pa = 0;
                    if (W > 0) {
                        pa = W - i[a];
                        if (i[a] - (n[a] - 1 - W) > pa) pa = i[a] - (n[a] - 1 - W);
                        if (pa < 0) pa = 0;
                    }
                    if (pa > p) p = pa;
                }
                const long cell = ((long)z * ny + y) * nx + x;
                if (p == 0) { mu_b[cell] = 0.0; inside[cell] = 1; }
                else {
                    const double delta = (double)p / (double)W;
                    mu_b[cell] = mu_lo + (mu_hi - mu_lo) * 0.5 * (1.0 - std::cos(PI * delta));
                    inside[cell] = 0;
                }
            }
}

// 1-D spectral derivative of every pencil of one field along `axis` (eq.(8),(10); R2, R5).
static void deriv_field(const double* f, double* df, int nx, int ny, int nz, int axis, double dx) {
    const int n[3] = {nx, ny, nz};
    const long st[3] = {1, nx, (long)nx * ny};
    const int na = n[axis];
    const int a1 = (axis + 1) % 3, a2 = (axis + 2) % 3;
    Dft fwd(na, -1), inv(na, +1);
    std::vector<double> k(na);
    wavenumbers(na, dx, k.data());
#pragma omp parallel
    {
        std::vector<cd> in(na), sp(na), out(na);
#pragma omp for collapse(2) schedule(static)
        for (int j2 = 0; j2 < n[a2]; ++j2)
            for (int j1 = 0; j1 < n[a1]; ++j1) {
                const long base = j1 * st[a1] + j2 * st[a2];
                for (int i = 0; i < na; ++i) in[i] = cd(f[base + i * st[axis]], 0.0);
                fwd.run(in.data(), 1, sp.data());
                for (int i = 0; i < na; ++i) sp[i] *= cd(0.0, k[i]);
                inv.run(sp.data(), 1, out.data());
                for (int i = 0; i < na; ++i) df[base + i * st[axis]] = out[i].real() / (double)na;
            }
    }
}

// d-dimensional DFT of one complex field, in place, by 1-D transforms along every axis (sign -1 fwd / +1 inverse,
// inverse normalised by 1/n per axis).
static void dft_nd(cd* f, int dim, int nx, int ny, int nz, int sign) {
    const int n[3] = {nx, ny, nz};
    const long st[3] = {1, nx, (long)nx * ny};
    for (int axis = 0; axis < dim; ++axis) {
        const int na = n[axis];
        const int a1 = (axis + 1) % 3, a2 = (axis + 2) % 3;
        Dft plan(na, sign);
#pragma omp parallel
        {
            std::vector<cd> in(na), out(na);
#pragma omp for collapse(2) schedule(static)
            for (int j2 = 0; j2 < n[a2]; ++j2)
                for (int j1 = 0; j1 < n[a1]; ++j1) {
                    const long base = j1 * st[a1] + j2 * st[a2];
                    for (int i = 0; i < na; ++i) in[i] = f[base + i * st[axis]];
                    plan.run(in.data(), 1, out.data());
                    const double sc = sign > 0 ? 1.0 / (double)na : 1.0;
                    for (int i = 0; i < na; ++i) f[base + i * st[axis]] = out[i] * sc;
                }
        }
    }
}

static double source_time(const Oracle* o, double t) {
    if (o->src_kind == 1) return 1.0;
    if (o->src_kind == 2) { const double u = (t - o->src_t0) / o->src_sigt; return std::exp(-0.5 * u * u); }
    return 0.0;
}

// streaming term T[c][cell] for the current state, formulation 1 (per-axis, real basis)
static void streaming_per_axis(const Oracle* o, std::vector<double>& T) {
    const int C = o->C; const long G = o->G;
    T.assign((size_t)C * G, 0.0);
    std::vector<double> d((size_t)G);
    for (int axis = 0; axis < o->dim; ++axis)
        for (int cp = 0; cp < C; ++cp) {
            bool used = false;
            for (int c = 0; c < C; ++c) if (o->A[axis][(size_t)c * C + cp] != 0.0) used = true;
            if (!used) continue;
            deriv_field(&o->psi[(size_t)cp * G], d.data(), o->nx, o->ny, o->nz, axis, o->dx);
            for (int c = 0; c < C; ++c) {
                const double w = o->A[axis][(size_t)c * C + cp];
                if (w == 0.0) continue;
                double* Tc = &T[(size_t)c * G];
#pragma omp parallel for schedule(static)
                for (long r = 0; r < G; ++r) Tc[r] += w * d[r];
            }
        }
}

// streaming term, formulation 0 (the paper's literal recipe): complex fields, full DFT, eq.(10)
static void streaming_literal(const Oracle* o, std::vector<double>& T) {
    const int C = o->C; const long G = o->G;
    // real -> complex basis (R6/R8)
    std::vector<cd> pc((size_t)C * G, cd(0, 0));
    for (int i = 0; i < C; ++i)
        for (int j = 0; j < C; ++j) {
            const cd u = o->U[(size_t)i * C + j];
            if (u == cd(0, 0)) continue;
            const double* src = &o->psi[(size_t)j * G];
            cd* dst = &pc[(size_t)i * G];
#pragma omp parallel for schedule(static)
            for (long r = 0; r < G; ++r) dst[r] += u * src[r];
        }
    for (int i = 0; i < C; ++i) dft_nd(&pc[(size_t)i * G], o->dim, o->nx, o->ny, o->nz, -1);
    // eq.(10) in k-space with d/dx_a -> + i k_a (R2)
    std::vector<double> kx(o->nx), ky(o->ny), kz(o->nz);
    wavenumbers(o->nx, o->dx, kx.data());
    wavenumbers(o->ny, o->dx, ky.data());
    if (o->dim == 3) wavenumbers(o->nz, o->dx, kz.data()); else kz.assign(o->nz, 0.0);
    std::vector<cd> tc((size_t)C * G, cd(0, 0));
    for (int i = 0; i < C; ++i)
        for (int j = 0; j < C; ++j) {
            const cd ax = o->Ac[0][(size_t)i * C + j], ay = o->Ac[1][(size_t)i * C + j],
                     az = o->dim == 3 ? o->Ac[2][(size_t)i * C + j] : cd(0, 0);
            if (ax == cd(0, 0) && ay == cd(0, 0) && az == cd(0, 0)) continue;
            const cd* src = &pc[(size_t)j * G];
            cd* dst = &tc[(size_t)i * G];
#pragma omp parallel for schedule(static)
            for (int z = 0; z < o->nz; ++z)
                for (int y = 0; y < o->ny; ++y)
                    for (int x = 0; x < o->nx; ++x) {
                        const long r = ((long)z * o->ny + y) * o->nx + x;
                        const cd ik = ax * cd(0, kx[x]) + ay * cd(0, ky[y]) + az * cd(0, kz[z]);
                        dst[r] += ik * src[r];
                    }
        }
    for (int i = 0; i < C; ++i) dft_nd(&tc[(size_t)i * G], o->dim, o->nx, o->ny, o->nz, +1);
    // complex -> real basis; the imaginary remainder is round-off for a real radiance
    T.assign((size_t)C * G, 0.0);
    for (int i = 0; i < C; ++i)
        for (int j = 0; j < C; ++j) {
            const cd u = o->Ui[(size_t)i * C + j];
            if (u == cd(0, 0)) continue;
            const cd* src = &tc[(size_t)j * G];
            double* dst = &T[(size_t)i * G];
#pragma omp parallel for schedule(static)
            for (long r = 0; r < G; ++r) dst[r] += (u * src[r]).real();
        }
}

// psi <- psi - c dt ( T + sigma_l psi ) + c dt q(t_src): one forward-Euler update of eq.(11) with the source sampled
// at an explicit time (the plain step samples it at t_n, R14; the Runge-Kutta stages below at their stage times)
static void euler_update(Oracle* o, int formulation, double t_src) {
    const int C = o->C; const long G = o->G;
    std::vector<double> T;
    if (formulation == 0) streaming_literal(o, T); else streaming_per_axis(o, T);
    const double cdt = o->c * o->dt;
    const double ft = source_time(o, t_src);
    o->psi_new.resize((size_t)C * G);
    for (int c = 0; c < C; ++c) {
        const int l = o->L[c];
        const double* p = &o->psi[(size_t)c * G];
        const double* t = &T[(size_t)c * G];
        double* pn = &o->psi_new[(size_t)c * G];
#pragma omp parallel for schedule(static)
        for (long r = 0; r < G; ++r) {
            double sigma;
            if (o->inside[r]) {
                double gl = 1.0;
                for (int j = 0; j < l; ++j) gl *= o->g[r];           // g^l by repeated multiplication (R16)
                sigma = o->mu_a[r] + o->mu_s[r] * (1.0 - gl);        // mu_t - mu_s g^l  (eq.(9), R4)
            } else sigma = o->mu_b[r];                               // eq.(12)
            pn[r] = p[r] - cdt * (t[r] + sigma * p[r]);              // eq.(11) with R3
        }
    }
    if (o->src_kind != 0 && ft != 0.0) {
        for (int c = 0; c < C; ++c) {
            if (o->src_w[c] == 0.0) continue;
            double* pn = &o->psi_new[(size_t)c * G];
            for (int bz = 0; bz < o->src_ext[2]; ++bz)
                for (int by = 0; by < o->src_ext[1]; ++by)
                    for (int bx = 0; bx < o->src_ext[0]; ++bx) {
                        const int x = o->src_org[0] + bx, y = o->src_org[1] + by, z = o->src_org[2] + bz;
                        const long r = ((long)z * o->ny + y) * o->nx + x;
                        if (!o->inside[r]) continue;                 // q = 0 in the PML (eq.(12))
                        const double S = o->src_S[((size_t)bz * o->src_ext[1] + by) * o->src_ext[0] + bx];
                        pn[r] += cdt * o->src_w[c] * S * ft;
                    }
        }
    }
    o->psi.swap(o->psi_new);
}

static void one_step(Oracle* o, int formulation) {
    euler_update(o, formulation, (double)o->step_count * o->dt);   // R14: q at t_n
    o->step_count += 1;
}

// SURVEY §8(f2), NOT the paper's integrator (the paper uses forward Euler, eq.(11)): the three-stage, third-order
// strong-stability-preserving Runge-Kutta scheme of Shu & Osher written as convex combinations of Euler updates
// E(u; t) = u + dt F(u, t) of the same semi-discrete system eq.(9):
//     u1      = E(u^n; t_n)
//     u2      = 3/4 u^n + 1/4 E(u1; t_n + dt)
//     u^{n+1} = 1/3 u^n + 2/3 E(u2; t_n + dt/2)
// For u' = M u it gives u^{n+1} = (I + z + z^2/2 + z^3/6) u^n, z = dt M (pinned in tests/test_oracle_pins.py); its
// stability region contains |Im z| <= sqrt(3), so the skew-adjoint streaming operator no longer needs the scattering
// damping to be stable and dt can approach dx/c (R10).
static void one_step_ssprk3(Oracle* o, int formulation) {
    const size_t n = o->psi.size();
    const double tn = (double)o->step_count * o->dt;
    const std::vector<double> u0 = o->psi;
    euler_update(o, formulation, tn);                                   // psi = u1
    euler_update(o, formulation, tn + o->dt);                           // psi = E(u1)
    for (size_t i = 0; i < n; ++i) o->psi[i] = 0.75 * u0[i] + 0.25 * o->psi[i];          // u2
    euler_update(o, formulation, tn + 0.5 * o->dt);                     // psi = E(u2)
    for (size_t i = 0; i < n; ++i) o->psi[i] = u0[i] / 3.0 + (2.0 / 3.0) * o->psi[i];    // u^{n+1}
    o->step_count += 1;
}

// ------------------------------------------------------------------------------------------------------------
// the steady-state operator, a Krylov solve with it, and the exponential (integrating-factor) step.
// PAPER.md:109 ("...related to the method of exponential integrators.  Krylov subspace iterative methods can then be
// employed to find a steady-state solution through repeated application of the implicit operator") and PAPER.md:195.
// ------------------------------------------------------------------------------------------------------------
// sigma_l(r) of eq.(9)/(12): mu_a + mu_s (1 - g^l) in Omega, mu_b in the layer
static double sigma_of(const Oracle* o, int l, long r) {
    if (!o->inside[r]) return o->mu_b[r];
    double gl = 1.0;
    for (int j = 0; j < l; ++j) gl *= o->g[r];
    return o->mu_a[r] + o->mu_s[r] * (1.0 - gl);
}

// The time-independent transport operator of eq.(9) with d/dt = 0:   (L psi)_c = T_c[psi] + sigma_l psi_c,
// so that eq.(9) reads  d psi/dt = -c L psi + c q  and a steady state satisfies  L psi = q.   y = L x, both [C][G].
static void apply_operator(Oracle* o, int formulation, const std::vector<double>& x, std::vector<double>& y) {
    const int C = o->C; const long G = o->G;
    std::vector<double> keep = x;          // the streaming routines read o->psi
    keep.swap(o->psi);
    std::vector<double> T;
    if (formulation == 0) streaming_literal(o, T); else streaming_per_axis(o, T);
    y.resize((size_t)C * G);
    for (int c = 0; c < C; ++c) {
        const int l = o->L[c];
#pragma omp parallel for schedule(static)
        for (long r = 0; r < G; ++r) y[(size_t)c * G + r] = T[(size_t)c * G + r] + sigma_of(o, l, r) * o->psi[(size_t)c * G + r];
    }
    keep.swap(o->psi);
}

// q_c(r) = w_c S(r) 1_Omega(r): the spatial/angular part of the source (temporal factor 1), [C][G]
static void source_field(const Oracle* o, std::vector<double>& q) {
    const int C = o->C; const long G = o->G;
    q.assign((size_t)C * G, 0.0);
    if (o->src_kind == 0) return;
    for (int c = 0; c < C; ++c)
        for (int bz = 0; bz < o->src_ext[2]; ++bz)
            for (int by = 0; by < o->src_ext[1]; ++by)
                for (int bx = 0; bx < o->src_ext[0]; ++bx) {
                    const int x = o->src_org[0] + bx, y = o->src_org[1] + by, z = o->src_org[2] + bz;
                    const long r = ((long)z * o->ny + y) * o->nx + x;
                    if (!o->inside[r]) continue;
                    q[(size_t)c * G + r] = o->src_w[c] * o->src_S[((size_t)bz * o->src_ext[1] + by) * o->src_ext[0] + bx];
                }
}

// Restarted GMRES(m) for L x = b (textbook: Saad, "Iterative methods for sparse linear systems", Alg. 6.9 — Arnoldi
// with modified Gram-Schmidt, Givens rotations on the Hessenberg matrix), plain Euclidean inner product, no
// preconditioner.  x holds the initial guess on entry and the solution on exit.  Stops when the TRUE residual
// ||b - L x|| / ||b|| (recomputed at every restart) is <= tol or after max_restarts cycles.  Returns the number of
// operator applications; *relres_out = the final true relative residual.
static long gmres_solve(Oracle* o, int formulation, const std::vector<double>& b, std::vector<double>& x, int m,
                        double tol, int max_restarts, double* relres_out) {
    const size_t n = b.size();
    auto dot = [&](const std::vector<double>& u, const std::vector<double>& v) {
        double s = 0;
#pragma omp parallel for reduction(+ : s) schedule(static)
        for (long i = 0; i < (long)n; ++i) s += u[i] * v[i];
        return s;
    };
    const double bnorm = std::sqrt(dot(b, b));
    long applications = 0;
    double relres = 0.0;
    if (bnorm == 0.0) { x.assign(n, 0.0); *relres_out = 0.0; return 0; }
    std::vector<std::vector<double>> V((size_t)m + 1);
    std::vector<double> H((size_t)(m + 1) * m), cs(m), sn(m), gv(m + 1), w, r;
    for (int cycle = 0; cycle <= max_restarts; ++cycle) {
        apply_operator(o, formulation, x, w); ++applications;
        r.resize(n);
        for (size_t i = 0; i < n; ++i) r[i] = b[i] - w[i];
        const double beta = std::sqrt(dot(r, r));
        relres = beta / bnorm;
        if (relres <= tol || cycle == max_restarts) break;
        V[0].resize(n);
        for (size_t i = 0; i < n; ++i) V[0][i] = r[i] / beta;
        std::fill(gv.begin(), gv.end(), 0.0);
        gv[0] = beta;
        int k = 0;
        for (; k < m; ++k) {
            apply_operator(o, formulation, V[k], w); ++applications;
            for (int j = 0; j <= k; ++j) {                       // modified Gram-Schmidt
                const double h = dot(w, V[j]);
                H[(size_t)j * m + k] = h;
                const double* vj = V[j].data();
#pragma omp parallel for schedule(static)
                for (long i = 0; i < (long)n; ++i) w[i] -= h * vj[i];
            }
            const double hn = std::sqrt(dot(w, w));
            H[(size_t)(k + 1) * m + k] = hn;
            for (int j = 0; j < k; ++j) {                        // earlier rotations on the new column
                const double a = H[(size_t)j * m + k], c2 = H[(size_t)(j + 1) * m + k];
                H[(size_t)j * m + k] = cs[j] * a + sn[j] * c2;
                H[(size_t)(j + 1) * m + k] = -sn[j] * a + cs[j] * c2;
            }
            const double a = H[(size_t)k * m + k], d = std::sqrt(a * a + hn * hn);
            cs[k] = a / d; sn[k] = hn / d;
            H[(size_t)k * m + k] = d; H[(size_t)(k + 1) * m + k] = 0.0;
            gv[k + 1] = -sn[k] * gv[k];
            gv[k] = cs[k] * gv[k];
            if (hn > 0) {
                V[k + 1].resize(n);
                for (size_t i = 0; i < n; ++i) V[k + 1][i] = w[i] / hn;
            }
            if (std::fabs(gv[k + 1]) / bnorm <= 0.1 * tol || hn == 0.0) { ++k; break; }
        }
        std::vector<double> yv(k);                               // back substitution  H y = g
        for (int i = k - 1; i >= 0; --i) {
            double s = gv[i];
            for (int j = i + 1; j < k; ++j) s -= H[(size_t)i * m + j] * yv[j];
            yv[i] = s / H[(size_t)i * m + i];
        }
        for (int j = 0; j < k; ++j) {
            const double* vj = V[j].data();
#pragma omp parallel for schedule(static)
            for (long i = 0; i < (long)n; ++i) x[i] += yv[j] * vj[i];
        }
    }
    *relres_out = relres;
    return applications;
}

// Exponential (integrating-factor) Euler step — SURVEY §8(f2), the family PAPER.md:109 points to; NOT eq.(11).
// The diagonal part of eq.(9), d psi/dt = -c sigma_l psi, is integrated exactly over the step and the streaming term
// explicitly (Lawson / integrating-factor Euler); the source enters through phi_1 so that a constant source is also
// integrated exactly where the streaming term vanishes:
//     psi_{n+1} = E ( psi_n - c dt T[psi_n] ) + Phi c dt q(t_n),     E = exp(-c dt sigma_l),  Phi = (1 - E)/(c dt sigma_l)
// (Phi = 1 where sigma_l = 0).  For a spatially uniform field (T = 0): psi(t_n) = e^{-c sigma_l t_n} psi(0)
// + (q/sigma_l)(1 - e^{-c sigma_l t_n}) with no O(dt) error — the pin.
static void one_step_exp(Oracle* o, int formulation) {
    const int C = o->C; const long G = o->G;
    std::vector<double> T;
    if (formulation == 0) streaming_literal(o, T); else streaming_per_axis(o, T);
    const double cdt = o->c * o->dt;
    const double ft = source_time(o, (double)o->step_count * o->dt);
    std::vector<double> q;
    source_field(o, q);
    o->psi_new.resize((size_t)C * G);
    for (int c = 0; c < C; ++c) {
        const int l = o->L[c];
#pragma omp parallel for schedule(static)
        for (long r = 0; r < G; ++r) {
            const size_t i = (size_t)c * G + r;
            const double a = cdt * sigma_of(o, l, r);
            const double E = std::exp(-a);
            const double Phi = a > 0 ? -std::expm1(-a) / a : 1.0;
            o->psi_new[i] = E * (o->psi[i] - cdt * T[i]) + Phi * cdt * ft * q[i];
        }
    }
    o->psi.swap(o->psi_new);
    o->step_count += 1;
}

// ------------------------------------------------------------------------------------------------------------
// C interface for the ctypes wrapper (oracle/rte_oracle.py)
// ------------------------------------------------------------------------------------------------------------
// One cell of one step, computed on its own (see orc_step_cell below).
template <typename Real>
static void step_cell_impl(void* h, const Real* psi, int x, int y, int z, double* out /*[C]*/) {
    Oracle* o = (Oracle*)h;
    const int C = o->C; const long G = o->G;
    const int n[3] = {o->nx, o->ny, o->nz};
    const long st[3] = {1, o->nx, (long)o->nx * o->ny};
    const int pos[3] = {x, y, z};
    const long cell = ((long)z * o->ny + y) * o->nx + x;
    std::vector<double> D((size_t)3 * C, 0.0);
    for (int a = 0; a < o->dim; ++a) {
        const int na = n[a];
        std::vector<double> k(na), d(na, 0.0);
        wavenumbers(na, o->dx, k.data());
        for (int r = 0; r < na; ++r) {
            double acc = 0;
            for (int q = 0; q < na; ++q) acc += -k[q] * std::sin(2.0 * PI * (double)((long)q * r % na) / (double)na);
            d[r] = acc / (double)na;
        }
        const long base = cell - pos[a] * st[a];
        for (int cp = 0; cp < C; ++cp) {
            double acc = 0;
            for (int j = 0; j < na; ++j) acc += d[((pos[a] - j) % na + na) % na] * (double)psi[(size_t)cp * G + base + j * st[a]];
            D[(size_t)a * C + cp] = acc;
        }
    }
    const double cdt = o->c * o->dt;
    const double ft = source_time(o, (double)o->step_count * o->dt);
    for (int c = 0; c < C; ++c) {
        double T = 0;
        for (int a = 0; a < o->dim; ++a)
            for (int cp = 0; cp < C; ++cp) T += o->A[a][(size_t)c * C + cp] * D[(size_t)a * C + cp];
        double sigma;
        if (o->inside[cell]) {
            double gl = 1.0;
            for (int j = 0; j < o->L[c]; ++j) gl *= o->g[cell];
            sigma = o->mu_a[cell] + o->mu_s[cell] * (1.0 - gl);
        } else sigma = o->mu_b[cell];
        const double p = (double)psi[(size_t)c * G + cell];
        double v = p - cdt * (T + sigma * p);
        if (o->src_kind != 0 && o->inside[cell]) {
            const int bx = x - o->src_org[0], by = y - o->src_org[1], bz = z - o->src_org[2];
            if (bx >= 0 && by >= 0 && bz >= 0 && bx < o->src_ext[0] && by < o->src_ext[1] && bz < o->src_ext[2])
                v += cdt * o->src_w[c] * o->src_S[((size_t)bz * o->src_ext[1] + by) * o->src_ext[0] + bx] * ft;
        }
        out[c] = v;
    }
}


extern "C" {

int orc_num_threads(void) {
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}
void orc_set_num_threads(int n) {
#ifdef _OPENMP
    omp_set_num_threads(n);
#else
    (void)n;
#endif
}

int orc_num_coeffs(int dim, int N) { return num_coeffs(dim, N); }

void orc_degrees(int dim, int N, int* L) {
    std::vector<int> v; degrees(dim, N, v);
    std::memcpy(L, v.data(), v.size() * sizeof(int));
}

// A[c*C + c'] : T_c = sum_c' A[c][c'] d_axis psi_c'.  Returns max |imag| of the transformed matrix.
double orc_coupling_real(int dim, int N, int axis, double* A) {
    std::vector<double> v;
    const double im = coupling_real(dim, N, axis, v);
    std::memcpy(A, v.data(), v.size() * sizeof(double));
    return im;
}

// complex-basis matrices of eq.(10) (3-D: index l*l+l+m; 2-D: m+N)
void orc_coupling_complex(int dim, int N, int axis, double* re, double* im) {
    std::vector<cd> Ax, Ay, Az;
    const int C = num_coeffs(dim, N);
    if (dim == 3) coupling_complex3(N, Ax, Ay, Az);
    else { coupling_complex2(N, Ax, Ay); Az.assign((size_t)C * C, cd(0, 0)); }
    const std::vector<cd>& A = axis == 0 ? Ax : (axis == 1 ? Ay : Az);
    for (size_t i = 0; i < A.size(); ++i) { re[i] = A[i].real(); im[i] = A[i].imag(); }
}

void orc_wavenumbers(int n, double dx, double* k) { wavenumbers(n, dx, k); }

void orc_dft(int n, int sign, const double* in_re, const double* in_im, double* out_re, double* out_im) {
    Dft plan(n, sign);
    std::vector<cd> a(n), b(n);
    for (int i = 0; i < n; ++i) a[i] = cd(in_re[i], in_im[i]);
    plan.run(a.data(), 1, b.data());
    for (int i = 0; i < n; ++i) { out_re[i] = b[i].real(); out_im[i] = b[i].imag(); }
}

void orc_deriv(const double* f, double* df, int nx, int ny, int nz, int axis, double dx) {
    deriv_field(f, df, nx, ny, nz, axis, dx);
}

void orc_pml_map(int dim, int nx, int ny, int nz, int W, double mu_lo, double mu_hi, double* mu_b,
                 unsigned char* inside) {
    pml_map(dim, nx, ny, nz, W, mu_lo, mu_hi, mu_b, inside);
}

// mu_a, mu_s, g: arrays of G doubles when *_is_map, else 1 value.
void* orc_create(int dim, int nx, int ny, int nz, int N, double dx, double dt, double c, const double* mu_a,
                 int mu_a_is_map, const double* mu_s, int mu_s_is_map, const double* g, int g_is_map, int pml_width,
                 double mu_lo, double mu_hi) {
    if (dim != 2 && dim != 3) return nullptr;
    if (dim == 2 && nz != 1) return nullptr;
    if (N < 1 || nx < 2 || ny < 2 || nz < 1 || dx <= 0 || dt <= 0 || c <= 0) return nullptr;
    Oracle* o = new Oracle();
    o->dim = dim; o->nx = nx; o->ny = ny; o->nz = nz; o->N = N; o->C = num_coeffs(dim, N);
    o->G = (long)nx * ny * nz; o->dx = dx; o->dt = dt; o->c = c;
    o->mu_a.resize(o->G); o->mu_s.resize(o->G); o->g.resize(o->G);
    for (long r = 0; r < o->G; ++r) {
        o->mu_a[r] = mu_a_is_map ? mu_a[r] : mu_a[0];
        o->mu_s[r] = mu_s_is_map ? mu_s[r] : mu_s[0];
        o->g[r] = g_is_map ? g[r] : g[0];
    }
    o->mu_b.resize(o->G); o->inside.resize(o->G);
    pml_map(dim, nx, ny, nz, pml_width, mu_lo, mu_hi, o->mu_b.data(), o->inside.data());
    degrees(dim, N, o->L);
    for (int a = 0; a < 3; ++a) coupling_real(dim, N, a, o->A[a]);
    {
        std::vector<cd> Ax, Ay, Az;
        if (dim == 3) coupling_complex3(N, Ax, Ay, Az);
        else { coupling_complex2(N, Ax, Ay); Az.assign((size_t)o->C * o->C, cd(0, 0)); }
        o->Ac[0] = Ax; o->Ac[1] = Ay; o->Ac[2] = Az;
    }
    basis_matrices(dim, N, o->U, o->Ui);
    o->psi.assign((size_t)o->C * o->G, 0.0);
    o->src_kind = 0; o->src_t0 = 0; o->src_sigt = 1; o->step_count = 0;
    for (int a = 0; a < 3; ++a) { o->src_org[a] = 0; o->src_ext[a] = 0; }
    return o;
}

void orc_destroy(void* h) { delete (Oracle*)h; }

void orc_set_state(void* h, const double* psi) {
    Oracle* o = (Oracle*)h;
    std::memcpy(o->psi.data(), psi, o->psi.size() * sizeof(double));
}
void orc_get_state(void* h, double* psi) {
    Oracle* o = (Oracle*)h;
    std::memcpy(psi, o->psi.data(), o->psi.size() * sizeof(double));
}
void orc_fluence(void* h, double* phi) {   // R9: coefficient 0
    Oracle* o = (Oracle*)h;
    std::memcpy(phi, o->psi.data(), (size_t)o->G * sizeof(double));
}
int orc_set_source(void* h, const double* w, const double* S, const int* origin, const int* extent, int kind,
                   double t0, double sigma_t) {
    Oracle* o = (Oracle*)h;
    const int n[3] = {o->nx, o->ny, o->nz};
    if (kind < 0 || kind > 2) return 1;
    if (kind == 2 && !(sigma_t > 0)) return 1;
    if (kind != 0)
        for (int a = 0; a < 3; ++a)
            if (origin[a] < 0 || extent[a] < 1 || origin[a] + extent[a] > n[a]) return 1;
    o->src_kind = kind; o->src_t0 = t0; o->src_sigt = sigma_t;
    if (kind == 0) return 0;
    o->src_w.assign(w, w + o->C);
    for (int a = 0; a < 3; ++a) { o->src_org[a] = origin[a]; o->src_ext[a] = extent[a]; }
    o->src_S.assign(S, S + (size_t)extent[0] * extent[1] * extent[2]);
    return 0;
}
void orc_step(void* h, int nsteps, int formulation) {
    Oracle* o = (Oracle*)h;
    for (int s = 0; s < nsteps; ++s) one_step(o, formulation);
}
void orc_step_ssprk3(void* h, int nsteps, int formulation) {
    Oracle* o = (Oracle*)h;
    for (int s = 0; s < nsteps; ++s) one_step_ssprk3(o, formulation);
}
double orc_time_ps(void* h) { Oracle* o = (Oracle*)h; return (double)o->step_count * o->dt; }

// streaming term only (no potential, no step): T[c][cell] of the current state
void orc_streaming(void* h, int formulation, double* T_out) {
    Oracle* o = (Oracle*)h;
    std::vector<double> T;
    if (formulation == 0) streaming_literal(o, T); else streaming_per_axis(o, T);
    std::memcpy(T_out, T.data(), T.size() * sizeof(double));
}

// One cell of one step, computed on its own (for sampled parity at sizes where a whole oracle step is too slow):
// psi_new[c] (all C) at cell (x,y,z) from the state psi ([C][nz][ny][nx], fp64), using the direct O(n) circulant
// sum of D_a along the three pencils through the cell:  (D_a f)[i] = sum_j d[(i-j) mod n] f[j],
// d[r] = (1/n) sum_k i k_a[k] exp(2 pi i k r / n)  (real, antisymmetric).
// One cell of one step, computed on its own (for sampled parity at sizes where a whole oracle step is too slow):
// psi_new[c] (all C) at cell (x,y,z) from the state psi ([C][nz][ny][nx]), using the direct O(n) circulant sum of D_a
// along the three pencils through the cell.  The _f32 variant reads an fp32 state (values promoted to fp64).
void orc_step_cell(void* h, const double* psi, int x, int y, int z, double* out) { step_cell_impl<double>(h, psi, x, y, z, out); }
void orc_step_cell_f32(void* h, const float* psi, int x, int y, int z, double* out) { step_cell_impl<float>(h, psi, x, y, z, out); }

// y = L x  (the steady-state operator above); x, y are [C][G]
void orc_apply_operator(void* h, int formulation, const double* x, double* y) {
    Oracle* o = (Oracle*)h;
    std::vector<double> xv(x, x + o->psi.size()), yv;
    apply_operator(o, formulation, xv, yv);
    std::memcpy(y, yv.data(), yv.size() * sizeof(double));
}
// q_c(r) = w_c S(r) 1_Omega(r), [C][G]
void orc_source_field(void* h, double* q) {
    Oracle* o = (Oracle*)h;
    std::vector<double> v;
    source_field(o, v);
    std::memcpy(q, v.data(), v.size() * sizeof(double));
}
// Steady state L psi = q by restarted GMRES(m) from the current state; the state becomes the solution.
// Returns the number of operator applications.
long orc_solve_steady(void* h, int formulation, int m, double tol, int max_restarts, double* relres_out) {
    Oracle* o = (Oracle*)h;
    std::vector<double> q;
    source_field(o, q);
    return gmres_solve(o, formulation, q, o->psi, m, tol, max_restarts, relres_out);
}
void orc_step_exp(void* h, int nsteps, int formulation) {
    Oracle* o = (Oracle*)h;
    for (int s = 0; s < nsteps; ++s) one_step_exp(o, formulation);
}

}  // extern "C"
