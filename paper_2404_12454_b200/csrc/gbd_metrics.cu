// gbd_metrics.cu -- figure of merit of the paper's beamlet-parameter search (Fig. 8-9), on the
// device: peak-normalised intensity I = |E|^2/|E0|^2 against the Airy pattern (2 J1(x)/x)^2,
// x = pi r/(lambda F#), as RMS difference over the whole detector and over the annular zones
// 0-5, 5-10, 10-15 lambda/D (R-13).  Deterministic two-stage reduction (no atomics).
#include <cstdio>
#include <mutex>

#include "gbd_common.cuh"

namespace {
constexpr int MT = 256;
constexpr int NACC = 9;   // sum d^2 and count for {all, zone0, zone1, zone2}, and max |d|

template <typename V2>
__global__ void __launch_bounds__(MT) metrics_partial_kernel(const V2 *__restrict__ field, int n_u, int n_v,
        double du, double dv, double inv_lfn, const double *__restrict__ e0, double *__restrict__ part)
{
    // blockIdx.y = run of a batched call: its own field, on-axis value and partial sums
    field += (size_t)blockIdx.y * n_u * n_v;
    e0 += 2 * blockIdx.y;
    part += (size_t)blockIdx.y * gridDim.x * NACC;
    __shared__ double sh[NACC][MT / 32];
    const double half_u = 0.5 * (double)(n_u - 1), half_v = 0.5 * (double)(n_v - 1);
    const double inv_i0 = 1.0 / (e0[0] * e0[0] + e0[1] * e0[1]);
    const double PI = 3.14159265358979323846;
    double acc[NACC];
#pragma unroll
    for (int k = 0; k < NACC; ++k) acc[k] = 0.0;
    const long n = (long)n_u * n_v;
    for (long idx = (long)blockIdx.x * MT + threadIdx.x; idx < n; idx += (long)gridDim.x * MT) {
        int iv = (int)(idx / n_u), iu = (int)(idx - (long)iv * n_u);
        double u = ((double)iu - half_u) * du, v = ((double)iv - half_v) * dv;
        double rl = sqrt(u * u + v * v) * inv_lfn;                 // radius in lambda F# (= lambda/D)
        double x = PI * rl;
        double a = 1.0;
        if (x != 0.0) { double t = 2.0 * j1(x) / x; a = t * t; }
        V2 e = field[idx];
        double d = ((double)e.x * (double)e.x + (double)e.y * (double)e.y) * inv_i0 - a;
        double d2 = d * d;
        acc[0] += d2; acc[1] += 1.0;
        int z = rl < 5.0 ? 0 : (rl < 10.0 ? 1 : (rl < 15.0 ? 2 : 3));
        if (z == 0) { acc[2] += d2; acc[3] += 1.0; }
        if (z == 1) { acc[4] += d2; acc[5] += 1.0; }
        if (z == 2) { acc[6] += d2; acc[7] += 1.0; }
        acc[8] = fmax(acc[8], fabs(d));
    }
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
#pragma unroll
    for (int k = 0; k < NACC; ++k) {
        double x = acc[k];
        for (int o = 16; o > 0; o >>= 1) {
            double y = __shfl_down_sync(0xffffffffu, x, o);
            x = (k == 8) ? fmax(x, y) : x + y;
        }
        if (lane == 0) sh[k][warp] = x;
    }
    __syncthreads();
    if (threadIdx.x < NACC) {
        int k = threadIdx.x;
        double x = sh[k][0];
        for (int w = 1; w < MT / 32; ++w) x = (k == 8) ? fmax(x, sh[k][w]) : x + sh[k][w];
        part[(long)blockIdx.x * NACC + k] = x;
    }
}

// out[0..3] = RMS over {all, 0-5, 5-10, 10-15 lambda/D}; out[4..7] = pixel counts; out[8] = max |I - Airy|
// One warp per accumulator: lane l adds the blocks l, l + 32, ... (independent loads in flight), then a fixed-order
// shuffle tree -- deterministic, and 2 us instead of the 55 us of one thread walking 592 dependent loads.
__global__ void __launch_bounds__(NACC * 32) metrics_final_kernel(const double *__restrict__ part, int nblocks,
                                                                  double *__restrict__ out, int out_stride,
                                                                  const long *__restrict__ counts)
{
    part += (size_t)blockIdx.x * nblocks * NACC;
    out += (size_t)blockIdx.x * out_stride;
    const int k = threadIdx.x >> 5, lane = threadIdx.x & 31;
    if (threadIdx.x == 0 && counts) out[9] = (double)counts[blockIdx.x];
    double x = 0.0;                                   // neutral for the sums and for the maximum of |d| >= 0
    for (int b = lane; b < nblocks; b += 32) {
        const double y = part[(long)b * NACC + k];
        x = (k == 8) ? fmax(x, y) : x + y;
    }
    for (int o = 16; o > 0; o >>= 1) {
        const double y = __shfl_down_sync(0xffffffffu, x, o);
        x = (k == 8) ? fmax(x, y) : x + y;
    }
    __shared__ double tot[NACC];
    if (lane == 0) tot[k] = x;
    __syncthreads();
    if (threadIdx.x < 4) {
        const int q = threadIdx.x;
        const double cnt = tot[2 * q + 1];
        out[q] = cnt > 0.0 ? sqrt(tot[2 * q] / cnt) : 0.0;
        out[4 + q] = cnt;
    }
    if (threadIdx.x == 0) out[8] = tot[8];
}
}  // namespace

int gbd_metrics_blocks(long n_px)
{
    long b = (n_px + MT - 1) / MT;
    return (int)(b < 1 ? 1 : (b > 592 ? 592 : b));
}

cudaError_t gbd_launch_metrics(const void *d_field, int precision, const gbd_detector &det, double lambda_fnum,
                               const double *d_e0, double *d_out, double *d_part, int n_runs, int out_stride,
                               const long *d_counts, cudaStream_t st)
{
    if (n_runs < 1) return cudaSuccess;
    dim3 nb(gbd_metrics_blocks((long)det.n_u * det.n_v), n_runs);
    if (precision == GBD_PRECISION_FP64)
        metrics_partial_kernel<double2><<<nb, MT, 0, st>>>((const double2 *)d_field, det.n_u, det.n_v, det.du,
                                                         det.dv, 1.0 / lambda_fnum, d_e0, d_part);
    else
        metrics_partial_kernel<float2><<<nb, MT, 0, st>>>((const float2 *)d_field, det.n_u, det.n_v, det.du,
                                                        det.dv, 1.0 / lambda_fnum, d_e0, d_part);
    cudaError_t e = cudaGetLastError();
    if (e != cudaSuccess) return e;
    metrics_final_kernel<<<n_runs, NACC * 32, 0, st>>>(d_part, (int)nb.x, d_out, out_stride, d_counts);
    return cudaGetLastError();
}

// ---------------------------------------------------------------------------------------------------------------
// gbd_psf_metrics_static: the figure of merit for callers that have no device memory to give as a workspace and no
// way of getting some (gbd.h says who they are).  The block partials of metrics_partial_kernel go to the array below
// instead: it is part of the library image, so every GPU that loads libgbd.so carries these bytes from the moment
// the module is loaded on it until the process exits, whether or not this entry point is ever called.
//
// Three things follow from one array serving every call:
//   - it is as large as it is and no larger: GBD_STATIC_METRICS_ROWS block rows, bigger requests are refused;
//   - it still holds whatever the previous call left there.  That is harmless here, and nothing is cleared:
//     metrics_partial_kernel stores all NACC values of every (field, block) row unconditionally and
//     metrics_final_kernel reads exactly those rows, so no value is ever read that the same call did not write;
//   - two calls whose kernels are on the GPU at the same time (different streams of one device, or two host threads)
//     write the same rows.  Calls on one stream are ordered and safe; anything else is the caller's to serialise.
namespace {
static __device__ __align__(256) double g_static_part[(size_t)GBD_STATIC_METRICS_ROWS * NACC];
static_assert(GBD_STATIC_METRICS_ROWS >= 592, "one field of any size must fit (gbd_metrics_blocks caps at 592)");

// `g_static_part` in HOST code is only a handle for the runtime's symbol table -- handing it to a kernel as if it
// were a pointer would make the kernel fault (or scribble over host memory on systems where the GPU can reach it).
// The device address comes from cudaGetSymbolAddress, differs from GPU to GPU, and is looked up once per device, the
// first time a call arrives with that device current.
constexpr int STATIC_MAX_DEVICES = 64;
std::mutex g_static_mutex;
double *g_static_addr[STATIC_MAX_DEVICES] = {};

cudaError_t static_part_address(double **out)
{
    int dev = -1;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) return e;
    if (dev < 0 || dev >= STATIC_MAX_DEVICES) return cudaErrorInvalidDevice;
    std::lock_guard<std::mutex> lock(g_static_mutex);
    if (!g_static_addr[dev]) {
        void *p = nullptr;
        e = cudaGetSymbolAddress(&p, g_static_part);     // resolves on the CURRENT device (loads the module there)
        if (e != cudaSuccess) return e;
        if (!p) return cudaErrorInvalidSymbol;
        g_static_addr[dev] = static_cast<double *>(p);
    }
    *out = g_static_addr[dev];
    return cudaSuccess;
}
}  // namespace

extern "C" gbd_status gbd_psf_metrics_static(const void *d_fields, int n_fields, int precision,
                                             const gbd_detector *det, double lambda_fnum, const double *d_e0,
                                             double *d_metrics, void *cuda_stream)
{
    if (!d_fields || !d_e0 || !d_metrics) return gbd_api_fail(GBD_EINVAL, "gbd_psf_metrics_static: null pointer");
    if (!gbd_api_detector_ok(det)) return gbd_api_fail(GBD_EINVAL, "gbd_psf_metrics_static: bad detector");
    if (precision != 0 && precision != 1)
        return gbd_api_fail(GBD_EINVAL, "gbd_psf_metrics_static: precision must be 0 or 1");
    if (!(lambda_fnum > 0.0)) return gbd_api_fail(GBD_EINVAL, "gbd_psf_metrics_static: lambda_fnum must be > 0");
    if (n_fields < 1) return gbd_api_fail(GBD_EINVAL, "gbd_psf_metrics_static: n_fields must be >= 1");
    const long rows = (long)n_fields * gbd_metrics_blocks((long)det->n_u * det->n_v);
    if (rows > (long)GBD_STATIC_METRICS_ROWS) {
        char msg[320];
        snprintf(msg, sizeof msg,
                 "gbd_psf_metrics_static: %d fields of %d x %d px need %ld block rows of scratch, the built-in array "
                 "holds %d (split the batch, or use gbd_psf_metrics with a workspace)",
                 n_fields, det->n_u, det->n_v, rows, (int)GBD_STATIC_METRICS_ROWS);
        return gbd_api_fail(GBD_ECAPACITY, msg);
    }
    double *d_part = nullptr;
    cudaError_t e = static_part_address(&d_part);
    if (e != cudaSuccess) return gbd_api_cuda_fail(e, "gbd_psf_metrics_static: address of the built-in scratch array");
    e = gbd_launch_metrics(d_fields, precision, *det, lambda_fnum, d_e0, d_metrics, d_part, n_fields, NACC, nullptr,
                           (cudaStream_t)cuda_stream);
    if (e != cudaSuccess) return gbd_api_cuda_fail(e, "gbd_psf_metrics_static: metrics kernels");
    return gbd_api_done((cudaStream_t)cuda_stream, 2, "gbd_psf_metrics_static (GBD_DEBUG_SYNC)");
}
