// cufft_literal.cu — the PAPER'S OWN GPU structure as a timed reference point; NOT the product.
//
// "A three-dimensional FFT is applied over the spatial dimensions of the complex valued input radiance
// field.  The directional gradient operator is then applied to the resulting k-space coefficients according to eq. (10).
// The solution is returned from k-space through application of an inverse transform.  2. The potential operators
// (mu_t - mu_s g^l) are applied to the input radiance field, and the result from (1) is added ... 3. time stepping is
// applied according to eq. (11) which updates the input radiance field in place ... a set of custom CUDA kernels ...
// the cuFFT library is used to implement the FFT."
//
// So: complex psi_l^m for all m in [-l, l] ((N+1)^2 complex fields, field-major [c][z][y][x]), one 3-D C2C cuFFT per
// field, one kernel for eq.(10) in k-space, one inverse cuFFT per field, one pointwise kernel for the potential and
// the forward-Euler update.  Same readings as the product (R1-R5): 1/(2l+1) on all three brackets, d/dx_a ->
// +i k_a, the Nyquist bin zeroed, psi^{n+1} = psi^n - c dt (T + sigma_l psi^n).  No source term (a source-free run is all
// the reference point needs).  It shares no code with paper_1801_06364_b200/ or oracle/.
#include <cuda_runtime.h>
#include <cufft.h>

#include <cmath>
#include <cstdio>
#include <vector>

namespace {

struct Entry { int src; int type; float coef; };   // type 0: i kz ; 1: -(i kx + ky)/2 ; 2: -(i kx - ky)/2   (times coef)

struct Ctx {
    int nx, ny, nz, N, C;
    long long G;
    float cdt;
    cudaStream_t stream;
    float2 *psi = nullptr, *hat = nullptr, *that = nullptr;
    const float *sa, *ss, *gm;
    Entry* entries = nullptr;     // [C][6]
    int* deg = nullptr;           // [C]
    float *kx = nullptr, *ky = nullptr, *kz = nullptr;
    cufftHandle plan = 0;
    size_t bytes = 0;
    long long launches = 0;
};

inline int cidx(int l, int m) { return l * l + l + m; }
inline double alpha(int l, int m) { const int v = (l + m) * (l - m); return v > 0 ? std::sqrt((double)v) : 0.0; }
inline double beta(int l, int m) { const int v = (l + m) * (l + m - 1); return v > 0 ? std::sqrt((double)v) : 0.0; }

// eq.(10), PAPER.md:98 (with R1): the six neighbours of (l, m)
void build_entries(int N, std::vector<Entry>& e, std::vector<int>& deg) {
    const int C = (N + 1) * (N + 1);
    e.assign((size_t)C * 6, Entry{0, 0, 0.f});
    deg.assign(C, 0);
    auto ok = [&](int l, int m) { return l >= 0 && l <= N && m >= -l && m <= l; };
    for (int l = 0; l <= N; ++l)
        for (int m = -l; m <= l; ++m) {
            const int c = cidx(l, m);
            deg[c] = l;
            const double f = 1.0 / (2.0 * l + 1.0);
            Entry* row = &e[(size_t)c * 6];
            int k = 0;
            auto put = [&](int l2, int m2, int type, double w) {
                if (ok(l2, m2) && w != 0.0) row[k++] = Entry{cidx(l2, m2), type, (float)(f * w)};
            };
            put(l + 1, m, 0, alpha(l + 1, m));
            put(l - 1, m, 0, alpha(l, m));
            put(l - 1, m - 1, 1, beta(l, m));
            put(l + 1, m - 1, 1, -beta(l + 1, -m + 1));
            put(l - 1, m + 1, 2, -beta(l, -m));
            put(l + 1, m + 1, 2, beta(l + 1, m + 1));
            for (; k < 6; ++k) row[k] = Entry{c, 0, 0.f};
        }
}

__global__ void k_kspace(float2* __restrict__ that, const float2* __restrict__ hat, const Entry* __restrict__ entries,
                         const float* __restrict__ kx, const float* __restrict__ ky, const float* __restrict__ kz, int C,
                         int nx, int ny, long long G) {
    for (long long cell = blockIdx.x * (long long)blockDim.x + threadIdx.x; cell < G; cell += (long long)gridDim.x * blockDim.x) {
        const int x = (int)(cell % nx);
        const long long r = cell / nx;
        const float qx = kx[x], qy = ky[(int)(r % ny)], qz = kz[(int)(r / ny)];
        // multipliers: i kz ; -(i kx + ky)/2 ; -(i kx - ky)/2
        const float2 mul[3] = {make_float2(0.f, qz), make_float2(-0.5f * qy, -0.5f * qx), make_float2(0.5f * qy, -0.5f * qx)};
        for (int c = 0; c < C; ++c) {
            float2 acc = make_float2(0.f, 0.f);
#pragma unroll
            for (int j = 0; j < 6; ++j) {
                const Entry en = entries[c * 6 + j];
                if (en.coef == 0.f) continue;
                const float2 v = hat[(size_t)en.src * G + cell];
                const float2 m = mul[en.type];
                acc.x += en.coef * (m.x * v.x - m.y * v.y);
                acc.y += en.coef * (m.x * v.y + m.y * v.x);
            }
            that[(size_t)c * G + cell] = acc;
        }
    }
}

// psi <- psi - c dt ( F^-1[T^]/G + sigma_l psi ),  sigma_l = sa + ss (1 - g^l)  (maps already carry the PML: sa = mu_b, ss = 0)
__global__ void k_pointwise(float2* __restrict__ psi, const float2* __restrict__ t, const float* __restrict__ sa,
                            const float* __restrict__ ss, const float* __restrict__ gm, const int* __restrict__ deg, int C,
                            long long G, float cdt, float invG) {
    for (long long cell = blockIdx.x * (long long)blockDim.x + threadIdx.x; cell < G; cell += (long long)gridDim.x * blockDim.x) {
        const float a = sa[cell], s = ss[cell], g = gm[cell];
        for (int c = 0; c < C; ++c) {
            float pw = 1.f;
            for (int l = deg[c]; l > 0; --l) pw *= g;
            const float sig = a + s * (1.f - pw);
            const size_t i = (size_t)c * G + cell;
            const float2 p = psi[i], tv = t[i];
            psi[i] = make_float2(p.x - cdt * (tv.x * invG + sig * p.x), p.y - cdt * (tv.y * invG + sig * p.y));
        }
    }
}

void wavenumbers(int n, float dx, std::vector<float>& k) {
    k.resize(n);
    for (int j = 0; j < n; ++j) {
        const int f = (2 * j < n) ? j : ((2 * j == n) ? 0 : j - n);
        k[j] = (float)(6.283185307179586476925286766559 * (double)f / ((double)n * (double)dx));
    }
}

template <typename T>
bool upload(T** dst, const std::vector<T>& v, Ctx* c) {
    if (cudaMalloc((void**)dst, v.size() * sizeof(T)) != cudaSuccess) return false;
    c->bytes += v.size() * sizeof(T);
    return cudaMemcpy(*dst, v.data(), v.size() * sizeof(T), cudaMemcpyHostToDevice) == cudaSuccess;
}

}  // namespace

extern "C" {

void cl_destroy(void* h) {
    Ctx* c = (Ctx*)h;
    if (!c) return;
    cudaStreamSynchronize(c->stream);
    if (c->plan) cufftDestroy(c->plan);
    cudaFree(c->psi); cudaFree(c->hat); cudaFree(c->that); cudaFree(c->entries); cudaFree(c->deg);
    cudaFree(c->kx); cudaFree(c->ky); cudaFree(c->kz);
    delete c;
}

// sa/ss/gm: device maps of nx*ny*nz floats (sa = mu_a in Omega | mu_b in the layer, ss = mu_s | 0, gm = g), caller-owned
int cl_create(void** out, int nx, int ny, int nz, int N, float dx, float dt, float cc, const float* sa, const float* ss,
              const float* gm, void* stream) {
    if (!out || nx < 2 || ny < 2 || nz < 2 || N < 1 || N > 31) return 1;
    Ctx* c = new Ctx();
    c->nx = nx; c->ny = ny; c->nz = nz; c->N = N; c->C = (N + 1) * (N + 1);
    c->G = (long long)nx * ny * nz; c->cdt = cc * dt; c->stream = (cudaStream_t)stream;
    c->sa = sa; c->ss = ss; c->gm = gm;
    const size_t field = (size_t)c->C * c->G * sizeof(float2);
    if (cudaMalloc((void**)&c->psi, field) != cudaSuccess || cudaMalloc((void**)&c->hat, field) != cudaSuccess ||
        cudaMalloc((void**)&c->that, field) != cudaSuccess) { cl_destroy(c); return 2; }
    c->bytes += 3 * field;
    cudaMemsetAsync(c->psi, 0, field, c->stream);
    std::vector<Entry> e; std::vector<int> deg;
    build_entries(N, e, deg);
    std::vector<float> kx, ky, kz;
    wavenumbers(nx, dx, kx); wavenumbers(ny, dx, ky); wavenumbers(nz, dx, kz);
    if (!upload(&c->entries, e, c) || !upload(&c->deg, deg, c) || !upload(&c->kx, kx, c) || !upload(&c->ky, ky, c) ||
        !upload(&c->kz, kz, c)) { cl_destroy(c); return 2; }
    if (cufftPlan3d(&c->plan, nz, ny, nx, CUFFT_C2C) != CUFFT_SUCCESS) { cl_destroy(c); return 3; }
    cufftSetStream(c->plan, c->stream);
    size_t ws = 0;
    cufftGetSize(c->plan, &ws);
    c->bytes += ws;
    *out = c;
    return 0;
}

int cl_set_state(void* h, const float2* psi_dev) {
    Ctx* c = (Ctx*)h;
    return cudaMemcpyAsync(c->psi, psi_dev, (size_t)c->C * c->G * sizeof(float2), cudaMemcpyDeviceToDevice, c->stream) != cudaSuccess;
}
int cl_get_state(void* h, float2* psi_dev) {
    Ctx* c = (Ctx*)h;
    return cudaMemcpyAsync(psi_dev, c->psi, (size_t)c->C * c->G * sizeof(float2), cudaMemcpyDeviceToDevice, c->stream) != cudaSuccess;
}

int cl_step(void* h, int nsteps) {
    Ctx* c = (Ctx*)h;
    const int blocks = 148 * 8;
    for (int s = 0; s < nsteps; ++s) {
        for (int f = 0; f < c->C; ++f)
            if (cufftExecC2C(c->plan, c->psi + (size_t)f * c->G, c->hat + (size_t)f * c->G, CUFFT_FORWARD) != CUFFT_SUCCESS) return 3;
        k_kspace<<<blocks, 128, 0, c->stream>>>(c->that, c->hat, c->entries, c->kx, c->ky, c->kz, c->C, c->nx, c->ny, c->G);
        for (int f = 0; f < c->C; ++f)
            if (cufftExecC2C(c->plan, c->that + (size_t)f * c->G, c->that + (size_t)f * c->G, CUFFT_INVERSE) != CUFFT_SUCCESS) return 3;
        k_pointwise<<<blocks, 128, 0, c->stream>>>(c->psi, c->that, c->sa, c->ss, c->gm, c->deg, c->C, c->G, c->cdt,
                                                   1.0f / (float)c->G);
        c->launches += 2;
    }
    return cudaGetLastError() != cudaSuccess;
}

unsigned long long cl_device_bytes(void* h) { return (unsigned long long)((Ctx*)h)->bytes; }
long long cl_own_kernel_launches(void* h) { return ((Ctx*)h)->launches; }
int cl_num_coeffs(void* h) { return ((Ctx*)h)->C; }

}  // extern "C"
