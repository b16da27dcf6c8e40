// mathtab.cu -- tables of fastmath.cuh (2^(j/64); c_j and -log c_j), computed once per device in long
// double on the host and kept in device memory; md_math_probe applies one of the device functions to
// an array so that tests can measure their accuracy (tests/test_gpu_math.py).
#include <cmath>
#include <mutex>

#include "common.cuh"
#include "fastmath.cuh"

namespace {
constexpr int MAX_DEV = 64;
double* g_tab[MAX_DEV];
std::mutex g_mu;

__global__ void k_math_probe(int fn, int64_t n, const double* __restrict__ in, double* __restrict__ out,
                             const double* __restrict__ gtab) {
    __shared__ __align__(16) double s_tab[fm::TAB_DOUBLES];
    const fm::Tab tb = fm::stage_tables(s_tab, gtab);
    __syncthreads();
    const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n) return;
    const double a = in[i];
    double r = 0.0, s, c;
    switch (fn) {
        case 0: r = fm::exp(a, tb); break;
        case 1: r = fm::log(a, tb); break;
        case 2: r = fm::rcp(a); break;
        case 3: r = fm::rsqrt(a); break;
        case 4: fm::sincos_0_pi(a, &s, &c); r = s; break;
        case 5: fm::sincos_0_pi(a, &s, &c); r = c; break;
    }
    out[i] = r;
}
}  // namespace

const double* md_math_tables() {
    int dev = 0;
    if (cudaGetDevice(&dev) != cudaSuccess || dev < 0 || dev >= MAX_DEV) return nullptr;
    std::lock_guard<std::mutex> lock(g_mu);
    if (g_tab[dev]) return g_tab[dev];
    double h[fm::TAB_DOUBLES];
    for (int j = 0; j < fm::EXP_N; ++j) h[j] = (double)exp2l((long double)j / fm::EXP_N);
    for (int j = 0; j < fm::LOG_N; ++j) {
        const long double centre = 1.0L + ((long double)j + 0.5L) / fm::LOG_N;
        const double c = (double)(1.0L / centre);
        h[fm::EXP_N + 2 * j] = c;
        h[fm::EXP_N + 2 * j + 1] = (double)(-logl((long double)c));
    }
    double* d = nullptr;
    if (cudaMalloc(&d, sizeof(h)) != cudaSuccess) { cudaGetLastError(); return nullptr; }
    if (cudaMemcpy(d, h, sizeof(h), cudaMemcpyHostToDevice) != cudaSuccess) { cudaFree(d); return nullptr; }
    g_tab[dev] = d;
    return d;
}

extern "C" int md_math_probe(int fn, int64_t n, const double* in, double* out, void* stream) {
    if (fn < 0 || fn > 5 || n < 0 || (n > 0 && (!in || !out))) return MD_ERR_ARG;
    if (n == 0) return MD_OK;
    const double* tab = md_math_tables();
    if (!tab) return MD_ERR_ALLOC;
    k_math_probe<<<(unsigned)((n + 255) / 256), 256, 0, (cudaStream_t)stream>>>(fn, n, in, out, tab);
    MD_CUDA_TRY(cudaGetLastError());
    return MD_OK;
}
