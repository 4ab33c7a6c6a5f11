// probes.cu — FP64 issue-rate microkernels behind sie_dfmp2_probe_fp64 (include/sie_dfmp2.h).
// They give bench.py the live denominator of the "tensor" roofline: MEASURED_PEAKS.json has no FP64 entry.
//   kind 0: register-resident DMMA.8x8x4 (mma.sync.m8n8k4.f64), 16 independent accumulator pairs per warp
//   kind 1: register-resident DFMA, 8 independent chains per thread
//   kind 2: shared-memory-fed DMMA with the fragment loads of mma_pipeline.cuh (64x32 warp tile, LDS.128 per fragment)
#include "sie_common.cuh"
#include "sie_internal.h"
#include "../../include/sie_dfmp2.h"

namespace sie {

constexpr int PROBE_THREADS = 256;

__global__ void __launch_bounds__(PROBE_THREADS) probe_dmma_kernel(int iters, double* __restrict__ sink) {
    double c[16][2];
#pragma unroll
    for (int k = 0; k < 16; ++k) c[k][0] = c[k][1] = 0.0;
    const double a = 1.0 + 1e-9 * threadIdx.x, b = 1.0 - 1e-9 * threadIdx.x;
    for (int it = 0; it < iters; ++it) {
#pragma unroll
        for (int k = 0; k < 16; ++k) dmma884(c[k][0], c[k][1], a, b);
    }
    double s = 0.0;
#pragma unroll
    for (int k = 0; k < 16; ++k) s += c[k][0] + c[k][1];
    if (s == 123.456) sink[0] = s;  // never true; keeps the loop alive
}

__global__ void __launch_bounds__(PROBE_THREADS) probe_dfma_kernel(int iters, double* __restrict__ sink) {
    double c[8];
#pragma unroll
    for (int k = 0; k < 8; ++k) c[k] = 1e-3 * k;
    const double a = 1.0 - 1e-12 * threadIdx.x, b = 1e-9;
    for (int it = 0; it < iters; ++it) {
#pragma unroll
        for (int k = 0; k < 8; ++k) c[k] = fma(c[k], a, b);
    }
    double s = 0.0;
#pragma unroll
    for (int k = 0; k < 8; ++k) s += c[k];
    if (s == 123.456) sink[0] = s;
}

// 8 warps as a 2 x 4 grid of 64 x 32 warp tiles over a [128 + 128][8] stage, like the pair mainloop.
__global__ void __launch_bounds__(PROBE_THREADS) probe_smem_dmma_kernel(int iters, double* __restrict__ sink) {
    __shared__ __align__(16) double stage[2][256 * 8];
    for (int i = threadIdx.x; i < 2 * 256 * 8; i += PROBE_THREADS) (&stage[0][0])[i] = 1e-6 * (i & 255);
    __syncthreads();
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31, g = lane >> 2, t = lane & 3;
    const int wm = warp & 1, wn = warp >> 1;
    double acc[8][4][2];
#pragma unroll
    for (int i = 0; i < 8; ++i)
#pragma unroll
        for (int j = 0; j < 4; ++j) acc[i][j][0] = acc[i][j][1] = 0.0;
    const int offA = (wm * 64 + g) * 8 + 2 * t, offB = 128 * 8 + (wn * 32 + g) * 8 + 2 * t;
    for (int it = 0; it < iters; ++it) {
        const double* s = stage[it & 1];
        double2 a[8], b[4];
#pragma unroll
        for (int i = 0; i < 8; ++i) a[i] = *reinterpret_cast<const double2*>(s + offA + i * 64);
#pragma unroll
        for (int j = 0; j < 4; ++j) b[j] = *reinterpret_cast<const double2*>(s + offB + j * 64);
#pragma unroll
        for (int i = 0; i < 8; ++i)
#pragma unroll
            for (int j = 0; j < 4; ++j) {
                dmma884(acc[i][j][0], acc[i][j][1], a[i].x, b[j].x);
                dmma884(acc[i][j][0], acc[i][j][1], a[i].y, b[j].y);
            }
    }
    double s = 0.0;
#pragma unroll
    for (int i = 0; i < 8; ++i)
#pragma unroll
        for (int j = 0; j < 4; ++j) s += acc[i][j][0] + acc[i][j][1];
    if (s == 123.456) sink[0] = s;
}

// Launches `kind` on `ctas_per_sm` x SMs CTAs, times it with events on `st` (synchronising), returns flop count.
int run_probe(int kind, int iters, int ctas_per_sm, int num_sms, double* sink, double* flops, float* ms, cudaStream_t st) {
    if (iters < 1 || ctas_per_sm < 1 || kind < 0 || kind > 2) return SIE_EINVAL;
    const int grid = num_sms * ctas_per_sm;
    cudaEvent_t e0, e1;
    cudaError_t e = cudaEventCreate(&e0);
    if (e != cudaSuccess) return set_cuda_error(e);
    e = cudaEventCreate(&e1);
    if (e != cudaSuccess) {
        cudaEventDestroy(e0);
        return set_cuda_error(e);
    }
    for (int rep = 0; rep < 2; ++rep) {  // first pass warms up (clocks, instruction cache), second is timed
        cudaEventRecord(e0, st);
        if (kind == 0) {
            probe_dmma_kernel<<<grid, PROBE_THREADS, 0, st>>>(iters, sink);
            *flops = (double)grid * (PROBE_THREADS / 32) * (double)iters * 16.0 * 512.0;
        } else if (kind == 1) {
            probe_dfma_kernel<<<grid, PROBE_THREADS, 0, st>>>(iters, sink);
            *flops = (double)grid * PROBE_THREADS * (double)iters * 8.0 * 2.0;
        } else {
            probe_smem_dmma_kernel<<<grid, PROBE_THREADS, 0, st>>>(iters, sink);
            *flops = (double)grid * (PROBE_THREADS / 32) * (double)iters * 64.0 * 512.0;
        }
        note_launch();
        cudaEventRecord(e1, st);
    }
    e = cudaEventSynchronize(e1);
    if (e == cudaSuccess) e = cudaGetLastError();
    if (e == cudaSuccess) e = cudaEventElapsedTime(ms, e0, e1);
    cudaEventDestroy(e0);
    cudaEventDestroy(e1);
    return e == cudaSuccess ? SIE_OK : set_cuda_error(e);
}

}  // namespace sie
