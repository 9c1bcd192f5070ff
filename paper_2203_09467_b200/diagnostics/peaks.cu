// peaks.cu -- DIAGNOSTICS: the two roofs that actually bound the step kernels on B200, measured (SURVEY 8(d):
// "measure it with an FMA micro-kernel before quoting an ALU fraction").
//   1. fp64 arithmetic: independent chains of DFMA (and, since libemx is built with -fmad=false, of DMUL + DADD
//      pairs) per thread, enough warps to fill every SM: thread-instructions per second.
//   2. L2 bandwidth at the footprint of the track store: a buffer that fits the 126 MB L2 is read (and copied)
//      over and over; the first pass, which comes from HBM, is not timed.
// Stand-alone program: nvcc -O3 -gencode arch=compute_100a,code=sm_100a peaks.cu -o peaks && ./peaks
// Prints one JSON object.  Built and run by paper_2203_09467_b200/diagnostics/peaks.py; never linked into libemx.
#include <cuda_runtime.h>
#include <cstdio>
#include <cstdlib>

#define CK(x)                                                                         \
    do {                                                                              \
        cudaError_t e_ = (x);                                                         \
        if (e_ != cudaSuccess) {                                                      \
            fprintf(stderr, "%s: %s\n", #x, cudaGetErrorString(e_));                  \
            exit(1);                                                                  \
        }                                                                             \
    } while (0)

constexpr int kChains = 8;     // independent dependency chains per thread
constexpr int kIters = 4096;   // loop trips; every trip issues kChains (x2 for the mul+add variant) instructions

__global__ void __launch_bounds__(256) k_dfma(double *out, double a, double b) {
    double v[kChains];
#pragma unroll
    for (int k = 0; k < kChains; ++k) v[k] = (double)(threadIdx.x + k);
    for (int it = 0; it < kIters; ++it) {
#pragma unroll
        for (int k = 0; k < kChains; ++k) v[k] = fma(v[k], a, b);
    }
    double s = 0.0;
#pragma unroll
    for (int k = 0; k < kChains; ++k) s += v[k];
    if (s == 12345.678) out[blockIdx.x * blockDim.x + threadIdx.x] = s;  // keeps the chains alive
}

__global__ void __launch_bounds__(256) k_dmul_dadd(double *out, double a, double b) {
    double v[kChains];
#pragma unroll
    for (int k = 0; k < kChains; ++k) v[k] = (double)(threadIdx.x + k);
    for (int it = 0; it < kIters; ++it) {
#pragma unroll
        for (int k = 0; k < kChains; ++k) v[k] = __dadd_rn(__dmul_rn(v[k], a), b);  // never contracted
    }
    double s = 0.0;
#pragma unroll
    for (int k = 0; k < kChains; ++k) s += v[k];
    if (s == 12345.678) out[blockIdx.x * blockDim.x + threadIdx.x] = s;
}

// grid-stride read of n double2 words, `reps` times; the sum keeps the loads alive
__global__ void __launch_bounds__(256) k_read(const double2 *p, size_t n, int reps, double *out) {
    double s = 0.0;
    const size_t stride = (size_t)gridDim.x * blockDim.x;
    for (int r = 0; r < reps; ++r)
        for (size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += stride) {
            const double2 v = p[i];
            s += v.x + v.y;
        }
    if (s == 12345.678) out[0] = s;
}
__global__ void __launch_bounds__(256) k_copy(const double2 *p, double2 *q, size_t n, int reps) {
    const size_t stride = (size_t)gridDim.x * blockDim.x;
    for (int r = 0; r < reps; ++r)
        for (size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += stride) q[i] = p[i];
}

static float time_ms(cudaEvent_t a, cudaEvent_t b) {
    float ms = 0.f;
    CK(cudaEventElapsedTime(&ms, a, b));
    return ms;
}

int main(int argc, char **argv) {
    const double footprint_mb = argc > 1 ? atof(argv[1]) : 95.0;  // the track store of 2^20 slots
    int dev = 0, sms = 0, khz = 0;
    CK(cudaGetDevice(&dev));
    CK(cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev));
    CK(cudaDeviceGetAttribute(&khz, cudaDevAttrClockRate, dev));
    cudaEvent_t e0, e1;
    CK(cudaEventCreate(&e0));
    CK(cudaEventCreate(&e1));
    double *out;
    CK(cudaMalloc(&out, sizeof(double) * 256 * 64 * sms));

    // ---- fp64 arithmetic: 8 blocks of 256 threads per SM (64 warps per SM), best of 5
    const int blocks = 8 * sms;
    double best_fma = 0.0, best_ma = 0.0;
    for (int rep = 0; rep < 6; ++rep) {
        CK(cudaEventRecord(e0));
        k_dfma<<<blocks, 256>>>(out, 1.0000001, 1e-9);
        CK(cudaEventRecord(e1));
        CK(cudaEventSynchronize(e1));
        const double inst = (double)blocks * 256 * kIters * kChains;
        const double r = inst / (time_ms(e0, e1) * 1e-3);
        if (rep && r > best_fma) best_fma = r;
        CK(cudaEventRecord(e0));
        k_dmul_dadd<<<blocks, 256>>>(out, 1.0000001, 1e-9);
        CK(cudaEventRecord(e1));
        CK(cudaEventSynchronize(e1));
        const double r2 = 2.0 * inst / (time_ms(e0, e1) * 1e-3);
        if (rep && r2 > best_ma) best_ma = r2;
    }

    // ---- L2: a buffer of footprint_mb read repeatedly; and half of it copied onto the other half
    const size_t n = (size_t)(footprint_mb * 1e6 / 16.0);
    double2 *buf;
    CK(cudaMalloc(&buf, n * sizeof(double2)));
    CK(cudaMemset(buf, 0, n * sizeof(double2)));
    const int reps = 20;
    double best_rd = 0.0, best_cp = 0.0;
    for (int rep = 0; rep < 4; ++rep) {
        k_read<<<16 * sms, 256>>>(buf, n, 1, out);  // warm: pulls the buffer into L2
        CK(cudaEventRecord(e0));
        k_read<<<16 * sms, 256>>>(buf, n, reps, out);
        CK(cudaEventRecord(e1));
        CK(cudaEventSynchronize(e1));
        const double r = (double)n * 16.0 * reps / (time_ms(e0, e1) * 1e-3) / 1e9;
        if (r > best_rd) best_rd = r;
        k_copy<<<16 * sms, 256>>>(buf, buf + n / 2, n / 2, 1);
        CK(cudaEventRecord(e0));
        k_copy<<<16 * sms, 256>>>(buf, buf + n / 2, n / 2, reps);
        CK(cudaEventRecord(e1));
        CK(cudaEventSynchronize(e1));
        const double c = (double)(n / 2) * 32.0 * reps / (time_ms(e0, e1) * 1e-3) / 1e9;  // read + written bytes
        if (c > best_cp) best_cp = c;
    }
    printf("{\"sms\": %d, \"sm_clock_mhz\": %.0f, \"fp64_dfma_tinst_per_s\": %.4e, \"fp64_tinst_per_s\": %.4e, "
           "\"fp64_tflops_fma\": %.2f, \"l2_footprint_mb\": %.1f, \"l2_read_gbs\": %.1f, \"l2_gbs\": %.1f}\n",
           sms, khz / 1e3, best_fma, best_ma, 2.0 * best_fma / 1e12, footprint_mb, best_rd, best_cp);
    return 0;
}
