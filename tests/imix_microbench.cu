// imix_microbench.cu -- test-only micro-benchmark (not product code): issues the instruction mix DESIGN.md 6.6
// counts for the Philox K = 4 multi-spin half-sweep, per 32 sites: 137 IMAD.WIDE.U32 + 160 LOP3 + 128 carry-chain
// adds (64 add.cc / addc pairs) + 72 IADD, with NO loads, stores (but one at the end) or update logic, in eight
// independent dependency chains per thread.  What it measures: the rate at which the SMs can issue that mix, i.e.
// the bound DESIGN 6.6 derives from the issue-slot model, as sites per nanosecond ("flips/ns").
#include <cstdint>
#include <cuda_runtime.h>

__global__ void __launch_bounds__(128) imix_kernel(uint32_t *out, uint32_t iters, uint32_t m0, uint32_t m1, uint32_t c0)
{
    uint32_t a[8], b[8];
#pragma unroll
    for (int j = 0; j < 8; j++) a[j] = threadIdx.x * 2654435761u + j * 40503u + blockIdx.x, b[j] = a[j] ^ c0;
    for (uint32_t it = 0; it < iters; it++) {
#pragma unroll
        for (int i = 0; i < 137; i++) { // 137 wide multiplies, each followed by the xor of its halves: 137 LOP3
            const int j = i & 7;
            uint64_t w;
            asm volatile("mul.wide.u32 %0, %1, %2;" : "=l"(w) : "r"(a[j]), "r"((i & 1) ? m1 : m0));
            uint32_t lo = (uint32_t)w, hi = (uint32_t)(w >> 32);
            asm volatile("lop3.b32 %0, %1, %2, %3, 0x96;" : "=r"(a[j]) : "r"(hi), "r"(lo), "r"(b[j]));
        }
#pragma unroll
        for (int i = 0; i < 23; i++) { // the other 23 LOP3
            const int j = i & 7;
            asm volatile("lop3.b32 %0, %1, %2, %3, 0xe8;" : "=r"(b[j]) : "r"(b[j]), "r"(a[j]), "r"(c0));
        }
#pragma unroll
        for (int i = 0; i < 64; i++) { // 64 two-instruction carry chains (the threshold compares)
            const int j = i & 7;
            uint32_t t;
            asm volatile("{ .reg .u32 s; sub.cc.u32 s, %1, %2; addc.u32 %0, %3, %3; }" : "=r"(t) : "r"(a[j]), "r"(b[(j + 1) & 7]), "r"(b[j]));
            b[j] = t;
        }
#pragma unroll
        for (int i = 0; i < 72; i++) { // 72 plain additions (key schedule, counters)
            const int j = i & 7;
            asm volatile("add.u32 %0, %1, %2;" : "=r"(a[j]) : "r"(a[j]), "r"(c0 + i));
        }
    }
    uint32_t r = 0;
#pragma unroll
    for (int j = 0; j < 8; j++) r ^= a[j] ^ b[j];
    if (r == 0x12345u) out[blockIdx.x * blockDim.x + threadIdx.x] = r; // keeps the chains alive
}

// runs `reps` launches of `blocks` CTAs x 128 threads x `iters` mix units; returns milliseconds per launch
extern "C" float imix_run(uint32_t blocks, uint32_t iters, int reps)
{
    uint32_t *out = nullptr;
    if (cudaMalloc(&out, (size_t)blocks * 128 * 4) != cudaSuccess) return -1.f;
    cudaEvent_t e0, e1;
    cudaEventCreate(&e0);
    cudaEventCreate(&e1);
    for (int i = 0; i < 3; i++) imix_kernel<<<blocks, 128>>>(out, iters, 0xD2511F53u, 0xCD9E8D57u, 0x9E3779B9u);
    cudaEventRecord(e0);
    for (int i = 0; i < reps; i++) imix_kernel<<<blocks, 128>>>(out, iters, 0xD2511F53u, 0xCD9E8D57u, 0x9E3779B9u);
    cudaEventRecord(e1);
    float ms = -1.f;
    if (cudaEventSynchronize(e1) == cudaSuccess && cudaGetLastError() == cudaSuccess) cudaEventElapsedTime(&ms, e0, e1);
    cudaEventDestroy(e0);
    cudaEventDestroy(e1);
    cudaFree(out);
    return ms < 0.f ? ms : ms / reps;
}
