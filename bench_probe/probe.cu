// probe.cu -- register-only instruction-rate probe (probe_alu_rate), built into its own bench-side
// library libdedisp_probe.so: it is a micro-benchmark, not part of the product ABI (include/dedisp.h).
// bench.py uses it to MEASURE the ALU roofline denominator on the device it is
// running on instead of trusting a spec sheet.
// Each kernel runs 8 independent dependency chains per thread, 2048 iterations of
// 8 ops, on 2 CTAs of 1024 threads per SM; results are folded and stored so that
// nothing is optimised away.
#include <cuda_runtime.h>
#include <stdint.h>

#define CHAINS 8
#define ITERS 2048

template <int WHICH>
__global__ void __launch_bounds__(1024) probe_kernel(uint32_t *out, uint32_t seed)
{
    uint32_t r[CHAINS];
    float f[CHAINS];
#pragma unroll
    for (int i = 0; i < CHAINS; ++i) {
        r[i] = seed * (threadIdx.x + 1) + i * 0x9e3779b9u;
        f[i] = (float)(r[i] & 1023);
    }
    uint32_t k = seed | 1u, m = seed * 7u + 3u;
    __shared__ __align__(16) uint32_t sh[8192];
    for (int i = threadIdx.x; i < 8192; i += blockDim.x) sh[i] = seed + i;
    __syncthreads();
    // conflict-free shared-memory reads: consecutive lanes read consecutive words (u32) / 16-byte vectors (v4)
    const uint32_t a32 = (uint32_t)__cvta_generic_to_shared(sh) + 4u * threadIdx.x;
    const uint32_t a128 = (uint32_t)__cvta_generic_to_shared(sh) + 16u * threadIdx.x;
    for (int it = 0; it < ITERS; ++it) {
#pragma unroll
        for (int i = 0; i < CHAINS; ++i) {
            if (WHICH == 0)  // IADD3
                asm volatile("add.u32 %0, %0, %1;" : "+r"(r[i]) : "r"(k));
            else if (WHICH == 1)  // LOP3 (majority)
                asm volatile("lop3.b32 %0, %0, %1, %2, 0xE8;" : "+r"(r[i]) : "r"(k), "r"(m));
            else if (WHICH == 2)  // SHF funnel
                asm volatile("shf.r.wrap.b32 %0, %0, %1, %2;" : "+r"(r[i]) : "r"(k), "r"(m));
            else if (WHICH == 3)  // FADD
                asm volatile("add.f32 %0, %0, %1;" : "+f"(f[i]) : "f"(1.5f));
            else if (WHICH == 4)  // IMAD
                asm volatile("mad.lo.u32 %0, %0, %1, %2;" : "+r"(r[i]) : "r"(k), "r"(m));
            else if (WHICH == 6) {  // LDS.32 (+ one XOR so that the load is used)
                uint32_t t;
                asm volatile("ld.volatile.shared.u32 %0, [%1];" : "=r"(t) : "r"(a32 + 128u * i + 4096u * (it & 3)) : "memory");
                r[i] ^= t;
            } else if (WHICH == 7) {  // LDS.128
                uint32_t t0, t1, t2, t3;
                asm volatile("ld.volatile.shared.v4.u32 {%0, %1, %2, %3}, [%4];"
                             : "=r"(t0), "=r"(t1), "=r"(t2), "=r"(t3) : "r"(a128 + 512u * i + 8192u * (it & 1)) : "memory");
                r[i] ^= t0 ^ t1 ^ t2 ^ t3;
            } else if (WHICH == 8)  // PRMT (byte permute)
                asm volatile("prmt.b32 %0, %0, %1, %2;" : "+r"(r[i]) : "r"(k), "r"(m));
            else if (WHICH == 9)  // DP4A
                asm volatile("dp4a.u32.u32 %0, %1, %2, %0;" : "+r"(r[i]) : "r"(k), "r"(m));
            else {  // alternate LOP3 (alu pipe) and IMAD (fma pipe)
                if (i & 1)
                    asm volatile("lop3.b32 %0, %0, %1, %2, 0x96;" : "+r"(r[i]) : "r"(k), "r"(m));
                else
                    asm volatile("mad.lo.u32 %0, %0, %1, %2;" : "+r"(r[i]) : "r"(k), "r"(m));
            }
        }
    }
    uint32_t acc = 0;
#pragma unroll
    for (int i = 0; i < CHAINS; ++i) acc ^= r[i] ^ __float_as_uint(f[i]);
    out[blockIdx.x * blockDim.x + threadIdx.x] = acc;
}

// which: 0 = IADD3 (u32 add), 1 = LOP3, 2 = SHF funnel shift, 3 = FADD, 4 = IMAD, 5 = LOP3+IMAD mix,
// 6 = conflict-free LDS.32 (+ XOR), 7 = conflict-free LDS.128 (+ 4 XOR), 8 = PRMT, 9 = DP4A.
// Writes lane-operations per second (warp instructions * 32 / s; for 6 and 7: lane-loads of 4 / 16 bytes).
// Returns 0, or 1 = bad argument, 2 = CUDA error.
extern "C" int probe_alu_rate(int which, double *lane_ops_per_s)
{
    if (!lane_ops_per_s || which < 0 || which > 9) return 1;
    int dev = 0, sms = 0;
    if (cudaGetDevice(&dev) != cudaSuccess) return 2;
    if (cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess)
        return 2;
    const int blocks = 2 * sms, threads = 1024;
    uint32_t *d = nullptr;
    if (cudaMalloc(&d, (size_t)blocks * threads * 4) != cudaSuccess) return 2;
    cudaEvent_t e0, e1;
    cudaEventCreate(&e0);
    cudaEventCreate(&e1);
    float best = 1e30f;
    for (int rep = 0; rep < 5; ++rep) {
        cudaEventRecord(e0, 0);
        switch (which) {
            case 0: probe_kernel<0><<<blocks, threads>>>(d, 12345u + rep); break;
            case 1: probe_kernel<1><<<blocks, threads>>>(d, 12345u + rep); break;
            case 2: probe_kernel<2><<<blocks, threads>>>(d, 12345u + rep); break;
            case 3: probe_kernel<3><<<blocks, threads>>>(d, 12345u + rep); break;
            case 4: probe_kernel<4><<<blocks, threads>>>(d, 12345u + rep); break;
            case 5: probe_kernel<5><<<blocks, threads>>>(d, 12345u + rep); break;
            case 6: probe_kernel<6><<<blocks, threads>>>(d, 12345u + rep); break;
            case 7: probe_kernel<7><<<blocks, threads>>>(d, 12345u + rep); break;
            case 8: probe_kernel<8><<<blocks, threads>>>(d, 12345u + rep); break;
            default: probe_kernel<9><<<blocks, threads>>>(d, 12345u + rep); break;
        }
        cudaEventRecord(e1, 0);
        if (cudaEventSynchronize(e1) != cudaSuccess) {
            cudaFree(d);
            return 2;
        }
        float ms = 0;
        cudaEventElapsedTime(&ms, e0, e1);
        if (rep > 0 && ms < best) best = ms;
    }
    cudaEventDestroy(e0);
    cudaEventDestroy(e1);
    cudaFree(d);
    const double ops = (double)blocks * threads * (double)ITERS * CHAINS;
    *lane_ops_per_s = ops / (best * 1e-3);
    return 0;
}
