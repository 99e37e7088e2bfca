// fp64_probe.cu -- include/hydro_probe.h: the FP64-pipe probe behind bench.py's ALU roofline.
// A library of its own (libhydro_probe_b200.so): nothing of the hydro path lives here and
// nothing of this lives in libhydro_b200.so.
#include "../../include/hydro_probe.h"

#include <cuda_runtime.h>

namespace {

// MODE 0: 8 independent DFMA chains per thread; MODE 1: the same with DADD/DMUL alternating (no
// FMA); MODE 2: every DFMA followed by one independent integer multiply-add, to see whether the
// other pipes issue under a busy FP64 pipe or wait for it.  out[] keeps the results alive.
template <int MODE>
__global__ void __launch_bounds__(256)
k_fp64_probe(double* out, int iters, double c0, double c1)
{
    double x[8];
    unsigned k[8];
#pragma unroll
    for (int q = 0; q < 8; ++q) { x[q] = c0 + (double)(threadIdx.x + q); k[q] = threadIdx.x * 8u + q; }
    for (int it = 0; it < iters; ++it) {
#pragma unroll
        for (int q = 0; q < 8; ++q) {
            if (MODE == 1) x[q] = (it & 1) ? __dmul_rn(x[q], c1) : __dadd_rn(x[q], c0);
            else x[q] = fma(x[q], c1, c0);
            if (MODE == 2) k[q] = k[q] * 1664525u + (unsigned)it;
        }
    }
    double s = 0.0;
    unsigned ks = 0;
#pragma unroll
    for (int q = 0; q < 8; ++q) { s += x[q]; ks += k[q]; }
    out[(size_t)blockIdx.x * blockDim.x + threadIdx.x] = s + (double)(ks & 1u);
}

}  // namespace

extern "C" int hydro_probe_fp64(double *rates_host)
{
    if (!rates_host) return -1;
    const int blocks = 148 * 8, threads = 256, iters = 8192;
    double *out = nullptr;
    cudaEvent_t e0, e1;
    if (cudaMalloc(&out, (size_t)blocks * threads * 8) != cudaSuccess) return -2;
    cudaEventCreate(&e0); cudaEventCreate(&e1);
    int rc = 0;
    for (int mode = 0; mode < 3 && rc == 0; ++mode) {
        float best = 1e30f;
        for (int rep = 0; rep < 4; ++rep) {           // first repetition warms up
            cudaEventRecord(e0);
            if (mode == 0) k_fp64_probe<0><<<blocks, threads>>>(out, iters, 1e-9, 0.999999);
            else if (mode == 1) k_fp64_probe<1><<<blocks, threads>>>(out, iters, 1e-9, 0.999999);
            else k_fp64_probe<2><<<blocks, threads>>>(out, iters, 1e-9, 0.999999);
            cudaEventRecord(e1);
            if (cudaEventSynchronize(e1) != cudaSuccess) { rc = -3; break; }
            float ms = 0.f;
            cudaEventElapsedTime(&ms, e0, e1);
            if (rep > 0 && ms < best) best = ms;
        }
        // FP64 thread-instructions per second (one DFMA = one instruction)
        rates_host[mode] = (double)blocks * threads * 8.0 * iters / (best * 1e-3);
    }
    cudaEventDestroy(e0); cudaEventDestroy(e1);
    cudaFree(out);
    return rc;
}
