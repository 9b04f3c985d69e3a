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

}  // namespace

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
