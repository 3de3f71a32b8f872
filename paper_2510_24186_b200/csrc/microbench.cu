// microbench.cu -- the roofline denominators of the fused MC step, measured on the device the library runs on
// (DESIGN.md section 7).  Reached through tridsk_debug_microbench; bench.py runs them in the same
// process as the timed workload and divides by what they return.  Nothing here is on the docking path.
//
//   TRIDSK_MB_FFMA    independent FFMA chains, 8 per thread         -> FP32 FMA rate          work = flops
//   TRIDSK_MB_FFMA2   the same with packed fma.rn.f32x2             -> packed FP32 FMA rate   work = flops
//   TRIDSK_MB_MUFU    independent ex2.approx chains                  -> XU (MUFU) rate         work = MUFU ops
//   TRIDSK_MB_L2_READ coalesced 16-byte reads of a buffer, repeated  -> streaming read rate    work = bytes
//                     (a buffer below the L2 size is L2-resident after the first pass)
//   TRIDSK_MB_GATHER  one 16-byte load per lane from a pseudo-random 32-byte sector of the buffer (what a trilinear
//                     lookup in the cell-packed grid does once per atom)  -> sector gather rate  work = 32-byte sectors * 32
#include "internal.h"

__global__ void __launch_bounds__(256) mb_ffma_kernel(float* out, int iters) {
    float a[8];
    const float x = 1.0f + 1e-7f * (float)threadIdx.x, y = 1e-9f * (float)blockIdx.x;
#pragma unroll
    for (int k = 0; k < 8; ++k) a[k] = (float)k;
    for (int i = 0; i < iters; ++i) {
#pragma unroll
        for (int r = 0; r < 8; ++r) {
#pragma unroll
            for (int k = 0; k < 8; ++k) a[k] = fmaf(a[k], x, y);
        }
    }
    float s = 0.f;
#pragma unroll
    for (int k = 0; k < 8; ++k) s += a[k];
    if (s == 12345.678f) out[0] = s;                        // keeps the chains alive
}

__global__ void __launch_bounds__(256) mb_ffma2_kernel(float* out, int iters) {
    unsigned long long a[8];
    const float x = 1.0f + 1e-7f * (float)threadIdx.x, y = 1e-9f * (float)blockIdx.x;
    unsigned long long xx, yy;
    asm("mov.b64 %0, {%1, %1};" : "=l"(xx) : "f"(x));
    asm("mov.b64 %0, {%1, %1};" : "=l"(yy) : "f"(y));
#pragma unroll
    for (int k = 0; k < 8; ++k) { const float v = (float)k; asm("mov.b64 %0, {%1, %1};" : "=l"(a[k]) : "f"(v)); }
    for (int i = 0; i < iters; ++i) {
#pragma unroll
        for (int r = 0; r < 8; ++r) {
#pragma unroll
            for (int k = 0; k < 8; ++k) asm volatile("fma.rn.f32x2 %0, %0, %1, %2;" : "+l"(a[k]) : "l"(xx), "l"(yy));
        }
    }
    unsigned long long s = 0;
#pragma unroll
    for (int k = 0; k < 8; ++k) s ^= a[k];
    if (s == 0x123456789abcdefULL) out[0] = 1.f;
}

__global__ void __launch_bounds__(256) mb_mufu_kernel(float* out, int iters) {
    float a[8];
#pragma unroll
    for (int k = 0; k < 8; ++k) a[k] = -1e-3f * (float)(k + 1) - 1e-6f * (float)threadIdx.x;
    for (int i = 0; i < iters; ++i) {
#pragma unroll
        for (int r = 0; r < 8; ++r) {
#pragma unroll
            for (int k = 0; k < 8; ++k) asm volatile("ex2.approx.ftz.f32 %0, %0;" : "+f"(a[k]));
        }
    }
    float s = 0.f;
#pragma unroll
    for (int k = 0; k < 8; ++k) s += a[k];
    if (s == 12345.678f) out[0] = s;
}

__global__ void __launch_bounds__(256) mb_l2_read_kernel(const float4* __restrict__ buf, size_t n_vec, int iters, float* out) {
    float s = 0.f;
    const size_t stride = (size_t)gridDim.x * blockDim.x, t0 = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
    for (int i = 0; i < iters; ++i) {
        for (size_t j = t0; j < n_vec; j += 4 * stride) {   // four independent loads in flight per thread
            float4 v[4];
#pragma unroll
            for (int k = 0; k < 4; ++k) {
                const size_t jj = j + k * stride;
                v[k] = jj < n_vec ? __ldcg(buf + jj) : make_float4(0.f, 0.f, 0.f, 0.f);
            }
#pragma unroll
            for (int k = 0; k < 4; ++k) s += v[k].x + v[k].w;
        }
    }
    if (s == 12345.678f) out[0] = s;
}

__global__ void __launch_bounds__(256) mb_gather_kernel(const float4* __restrict__ buf, unsigned n_sec, int iters, float* out) {
    // per lane a multiplicative-congruential walk over the 32-byte sectors; four independent loads in flight
    unsigned h = (blockIdx.x * blockDim.x + threadIdx.x) * 2654435761u + 12345u;
    float s = 0.f;
    for (int i = 0; i < iters; ++i) {
        float4 v[4];
#pragma unroll
        for (int k = 0; k < 4; ++k) {
            h = h * 1664525u + 1013904223u;
            const unsigned sec = (unsigned)(((unsigned long long)h * n_sec) >> 32);
            v[k] = __ldg(buf + 2 * (size_t)sec + (h & 1u));  // one of the sector's two 16-byte halves
        }
#pragma unroll
        for (int k = 0; k < 4; ++k) s += v[k].x + v[k].w;
    }
    if (s == 12345.678f) out[0] = s;
}

// Runs microbenchmark `which` once on stream s; *work = the units of work the launch did (see the table above).
cudaError_t launch_microbench(cudaStream_t s, int which, int sm_count, void* buf, size_t bytes, int iters, float* sink, double* work) {
    const int blocks = sm_count * 8, threads = 256;
    const double lanes = (double)blocks * threads;
    switch (which) {
        case TRIDSK_MB_FFMA:
            mb_ffma_kernel<<<blocks, threads, 0, s>>>(sink, iters);
            *work = lanes * iters * 64.0 * 2.0;
            break;
        case TRIDSK_MB_FFMA2:
            mb_ffma2_kernel<<<blocks, threads, 0, s>>>(sink, iters);
            *work = lanes * iters * 64.0 * 4.0;
            break;
        case TRIDSK_MB_MUFU:
            mb_mufu_kernel<<<blocks, threads, 0, s>>>(sink, iters);
            *work = lanes * iters * 64.0;
            break;
        case TRIDSK_MB_L2_READ: {
            const size_t n_vec = bytes / 16;
            mb_l2_read_kernel<<<blocks, threads, 0, s>>>((const float4*)buf, n_vec, iters, sink);
            *work = (double)n_vec * 16.0 * iters;
            break;
        }
        case TRIDSK_MB_GATHER: {
            const size_t n_sec = bytes / 32;
            if (n_sec == 0 || n_sec > 0xffffffffULL) return cudaErrorInvalidValue;
            mb_gather_kernel<<<blocks, threads, 0, s>>>((const float4*)buf, (unsigned)n_sec, iters, sink);
            *work = lanes * iters * 4.0 * 32.0;
            break;
        }
        default:
            return cudaErrorInvalidValue;
    }
    return cudaGetLastError();
}
