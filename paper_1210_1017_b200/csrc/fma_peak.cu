// Measurement helper ("the builder measures a register-resident FMA-chain peak on the
// box"): the FP32 rate this GPU sustains when nothing but fused multiply-adds are issued, with all
// operands in registers - the denominator the interaction kernel's "alu" roofline is read against,
// next to the nominal 148 SMs x 128 lanes x 2 flop x clock.  Two forms:
//   variant 0  scalar FFMA, 8 independent chains per thread
//   variant 1  packed FFMA2 (fma.rn.f32x2, two fp32 lanes per instruction - the form the interaction
//              kernel's pair term uses), 4 independent chains of 2 lanes per thread
// Not on the hot path.
#include "sph_internal.cuh"

namespace sph {

__device__ __forceinline__ unsigned long long pk2(float a, float b)
{
    unsigned long long r;
    asm("mov.b64 %0, {%1, %2};" : "=l"(r) : "f"(a), "f"(b));
    return r;
}
__device__ __forceinline__ void upk2(unsigned long long v, float &a, float &b)
{
    asm("mov.b64 {%0, %1}, %2;" : "=f"(a), "=f"(b) : "l"(v));
}

template <int VARIANT>
__global__ void __launch_bounds__(256)
fma_peak_kernel(int iters, float seed, float *__restrict__ sink)
{
    const float a = 1.0f + seed * (float)(threadIdx.x & 7), b = seed;
    float r = 0.f;
    if (VARIANT == 0) {
        float x[8];
#pragma unroll
        for (int k = 0; k < 8; ++k) x[k] = (float)k * seed;
        for (int i = 0; i < iters; ++i) {
#pragma unroll
            for (int u = 0; u < 8; ++u) {
#pragma unroll
                for (int k = 0; k < 8; ++k) x[k] = fmaf(x[k], a, b);
            }
        }
#pragma unroll
        for (int k = 0; k < 8; ++k) r += x[k];
    } else {
        unsigned long long x[4];
        const unsigned long long a2 = pk2(a, a), b2 = pk2(b, b);
#pragma unroll
        for (int k = 0; k < 4; ++k) x[k] = pk2((float)k * seed, (float)(k + 4) * seed);
        for (int i = 0; i < iters; ++i) {
#pragma unroll
            for (int u = 0; u < 8; ++u) {
#pragma unroll
                for (int k = 0; k < 4; ++k)
                    asm volatile("fma.rn.f32x2 %0, %0, %1, %2;" : "+l"(x[k]) : "l"(a2), "l"(b2));
            }
        }
#pragma unroll
        for (int k = 0; k < 4; ++k) { float lo, hi; upk2(x[k], lo, hi); r += lo + hi; }
    }
    if (r == 123456.789f) sink[0] = r;          // never true for the seeds used; keeps the chains alive
}

// flops per launch = 2 (fma) x 8 lanes x 8 unrolled x iters x 256 threads x blocks
cudaError_t launch_fma_peak(sph_ctx *c, int variant, int iters, int blocks, float *sink)
{
    if (variant == 0) fma_peak_kernel<0><<<blocks, 256, 0, c->stream>>>(iters, 1e-3f, sink);
    else fma_peak_kernel<1><<<blocks, 256, 0, c->stream>>>(iters, 1e-3f, sink);
    c->n_launches++;
    return cudaGetLastError();
}

}  // namespace sph
