// Test helper (NOT product, NOT oracle): runs cuRAND's own device implementations of XORWOW and
// Philox4x32-10 from the toolkit headers on caller-given states, so that the ORACLE's recurrences and
// constants -- which PAPER.md does not print (readings R-B1, R-C1 come from Refs.[30],[20]) -- are
// pinned to an implementation that shares nothing with this repository.  curand_init's seeding
// scramble is bypassed on purpose: the state fields are set directly.
#include <cstdint>
#include <cuda_runtime.h>
#include <curand_kernel.h>

__global__ void cc_xorwow_kernel(const uint32_t *st, uint32_t n, uint32_t draws, uint32_t *out)
{
    const uint32_t i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n) return;
    curandStateXORWOW_t s;
    for (int k = 0; k < 5; k++) s.v[k] = st[6 * i + k]; // x, y, z, w, v
    s.d = st[6 * i + 5];
    s.boxmuller_flag = 0;
    s.boxmuller_flag_double = 0;
    s.boxmuller_extra = 0.f;
    s.boxmuller_extra_double = 0.;
    for (uint32_t j = 0; j < draws; j++) out[i * draws + j] = curand(&s);
}

__global__ void cc_philox_kernel(const uint32_t *ck, uint32_t n, uint32_t *out)
{
    const uint32_t i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n) return;
    const uint4 c = make_uint4(ck[6 * i], ck[6 * i + 1], ck[6 * i + 2], ck[6 * i + 3]);
    const uint2 k = make_uint2(ck[6 * i + 4], ck[6 * i + 5]);
    const uint4 r = curand_Philox4x32_10(c, k);
    out[4 * i] = r.x, out[4 * i + 1] = r.y, out[4 * i + 2] = r.z, out[4 * i + 3] = r.w;
}

template <class F>
static int run(const uint32_t *h_in, size_t in_words, uint32_t *h_out, size_t out_words, F launch)
{
    uint32_t *d_in = nullptr, *d_out = nullptr;
    if (cudaMalloc(&d_in, in_words * 4) != cudaSuccess || cudaMalloc(&d_out, out_words * 4) != cudaSuccess) return -1;
    cudaMemcpy(d_in, h_in, in_words * 4, cudaMemcpyHostToDevice);
    launch(d_in, d_out);
    const cudaError_t e = cudaMemcpy(h_out, d_out, out_words * 4, cudaMemcpyDeviceToHost);
    cudaFree(d_in);
    cudaFree(d_out);
    return e == cudaSuccess ? 0 : -2;
}

extern "C" int cc_xorwow(const uint32_t *h_states, uint32_t n, uint32_t draws, uint32_t *h_out)
{
    return run(h_states, (size_t)n * 6, h_out, (size_t)n * draws, [&](uint32_t *di, uint32_t *dout) {
        cc_xorwow_kernel<<<(n + 127) / 128, 128>>>(di, n, draws, dout);
    });
}

extern "C" int cc_philox(const uint32_t *h_ctr_key, uint32_t n, uint32_t *h_out)
{
    return run(h_ctr_key, (size_t)n * 6, h_out, (size_t)n * 4, [&](uint32_t *di, uint32_t *dout) {
        cc_philox_kernel<<<(n + 127) / 128, 128>>>(di, n, dout);
    });
}
