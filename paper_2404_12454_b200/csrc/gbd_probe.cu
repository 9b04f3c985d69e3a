// gbd_probe.cu -- FP64-pipe peak probe (roofline denominator measured on the box).
#include "gbd_common.cuh"

namespace {
constexpr int PROBE_THREADS = 256;
constexpr int PROBE_CHAINS = 8;
constexpr int PROBE_UNROLL = 16;

__global__ void __launch_bounds__(PROBE_THREADS) dfma_probe_kernel(double *sink, long iters, double seed)
{
    double a[PROBE_CHAINS];
#pragma unroll
    for (int c = 0; c < PROBE_CHAINS; ++c) a[c] = seed + (double)(threadIdx.x + c) * 1e-9;
    const double m = 0.999999999, k = 1e-12;
    for (long i = 0; i < iters; ++i) {
#pragma unroll
        for (int r = 0; r < PROBE_UNROLL; ++r) {
#pragma unroll
            for (int c = 0; c < PROBE_CHAINS; ++c) a[c] = fma(a[c], m, k);
        }
    }
    double s = 0.0;
#pragma unroll
    for (int c = 0; c < PROBE_CHAINS; ++c) s += a[c];
    if (s == 123456.789) *sink = s;            // never true; keeps the chains alive
}

// Variants used to characterise the FP64 pipe (profiles/r1_fp64_pipe_probes.md):
//   1: DFMA whose addend comes from the constant bank (2 register sources instead of 3)
//   2: 8 DFMA chains + one XOR and one ADD on the ALU pipe per 2 DFMAs
//   3: ONE dependent chain per thread (launch with 1 warp per SM sub-partition -> latency)
__constant__ double c_probe_k = 1e-12;
template <int MODE>
__global__ void __launch_bounds__(PROBE_THREADS) fp64_probe_kernel(double *sink, long iters, double seed,
                                                                  int sel)
{
    double a[PROBE_CHAINS];
    int q[PROBE_CHAINS];
#pragma unroll
    for (int c = 0; c < PROBE_CHAINS; ++c) {
        a[c] = seed + (double)(threadIdx.x + c) * 1e-9;
        q[c] = threadIdx.x * (c + 1);
    }
    const double m = 0.999999999;
    long long t0 = clock64();
    for (long i = 0; i < iters; ++i) {
#pragma unroll
        for (int r = 0; r < PROBE_UNROLL; ++r) {
            if (MODE == 3) {
                a[0] = fma(a[0], m, seed);
            } else {
#pragma unroll
                for (int c = 0; c < PROBE_CHAINS; ++c) {
                    a[c] = fma(a[c], m, MODE == 1 ? c_probe_k : seed);
                    if (MODE == 2 && (c & 1)) q[c] = (q[c] ^ sel) + 0x1234;
                }
            }
        }
    }
    long long t1 = clock64();
    double s = 0.0;
    int t = 0;
#pragma unroll
    for (int c = 0; c < PROBE_CHAINS; ++c) { s += a[c]; t += q[c]; }
    if (s == 123456.789 || t == -77) sink[0] = s + t;
    if (MODE == 3 && blockIdx.x == 0 && threadIdx.x == 0)
        sink[1] = (double)(t1 - t0) / ((double)iters * PROBE_UNROLL);      // cycles per dependent DFMA
}
}  // namespace

cudaError_t gbd_launch_probe_mode(int mode, double *d_sink, long iters, double *inst_per_launch, cudaStream_t st)
{
    int dev = 0, sms = 148;
    if (cudaGetDevice(&dev) == cudaSuccess)
        cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
    int blocks = sms * 8, threads = PROBE_THREADS;
    double per_thread = (double)PROBE_CHAINS * PROBE_UNROLL * (double)iters;
    switch (mode) {
    case 0: dfma_probe_kernel<<<blocks, threads, 0, st>>>(d_sink, iters, 1.0); break;
    case 1: fp64_probe_kernel<1><<<blocks, threads, 0, st>>>(d_sink, iters, 1e-12, 5); break;
    case 2: fp64_probe_kernel<2><<<blocks, threads, 0, st>>>(d_sink, iters, 1e-12, 5); break;
    case 3:
        blocks = sms; threads = 128; per_thread = (double)PROBE_UNROLL * (double)iters;
        fp64_probe_kernel<3><<<blocks, threads, 0, st>>>(d_sink, iters, 1e-12, 5);
        break;
    default: return cudaErrorInvalidValue;
    }
    if (inst_per_launch) *inst_per_launch = (double)blocks * threads * per_thread;
    return cudaGetLastError();
}

cudaError_t gbd_launch_probe(double *d_sink, long iters, double *dfma_per_launch, cudaStream_t st)
{
    int dev = 0, sms = 148;
    if (cudaGetDevice(&dev) == cudaSuccess)
        cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
    int blocks = sms * 8;
    dfma_probe_kernel<<<blocks, PROBE_THREADS, 0, st>>>(d_sink, iters, 1.0);
    if (dfma_per_launch)
        *dfma_per_launch = (double)blocks * PROBE_THREADS * PROBE_CHAINS * PROBE_UNROLL * (double)iters;
    return cudaGetLastError();
}
