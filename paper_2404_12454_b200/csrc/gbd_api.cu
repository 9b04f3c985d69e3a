// gbd_api.cu -- the C ABI of libgbd.so (include/gbd.h): argument validation, workspace carving, launches.
#include <atomic>
#include <cmath>
#include <cstdlib>
#include <cstdarg>
#include <cstdio>
#include <cstring>
#include <mutex>
#include <new>
#include <vector>

#include "gbd_common.cuh"

struct gbd_beamlets {
    long n;
    double waist, wavelength;
    bool propagated;
};

namespace {

thread_local char g_err[512] = "";
std::atomic<long> g_launches{0};
thread_local cudaEvent_t g_ev0 = nullptr, g_ev1 = nullptr;

// Pinned staging buffer for the small host tables of gbd_airy_sweep.  cudaMemcpyAsync from pageable memory makes
// the host wait for the stream's earlier work; from this buffer the upload is a plain stream-ordered DMA.  The
// buffer is reused by the next call, which waits (host side) only if that upload has not finished yet.
struct Staging {
    char *h = nullptr;
    size_t cap = 0;
    cudaEvent_t done = nullptr;
    int device = -1;
};
std::mutex g_stage_mutex;
Staging g_stage;

struct Upload { void *dst; const void *src; size_t bytes; };

cudaError_t staged_upload(const Upload *u, int n, cudaStream_t st)
{
    std::lock_guard<std::mutex> lock(g_stage_mutex);
    size_t total = 0;
    for (int i = 0; i < n; ++i) total += (u[i].bytes + 255) / 256 * 256;
    int dev = 0;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) return e;
    if (g_stage.done && (g_stage.device != dev || g_stage.cap < total)) {
        cudaEventSynchronize(g_stage.done);
        cudaEventDestroy(g_stage.done);
        cudaFreeHost(g_stage.h);
        g_stage = Staging();
    }
    if (!g_stage.h) {
        size_t cap = total < 65536 ? 65536 : total;
        e = cudaHostAlloc((void **)&g_stage.h, cap, cudaHostAllocPortable);
        if (e != cudaSuccess) { g_stage = Staging(); return e; }
        e = cudaEventCreateWithFlags(&g_stage.done, cudaEventDisableTiming);
        if (e != cudaSuccess) { cudaFreeHost(g_stage.h); g_stage = Staging(); return e; }
        g_stage.cap = cap;
        g_stage.device = dev;
    } else {
        e = cudaEventSynchronize(g_stage.done);          // previous upload out of the buffer (usually long done)
        if (e != cudaSuccess) return e;
    }
    size_t off = 0;
    for (int i = 0; i < n; ++i) {
        memcpy(g_stage.h + off, u[i].src, u[i].bytes);
        e = cudaMemcpyAsync(u[i].dst, g_stage.h + off, u[i].bytes, cudaMemcpyHostToDevice, st);
        if (e != cudaSuccess) return e;
        off += (u[i].bytes + 255) / 256 * 256;
    }
    return cudaEventRecord(g_stage.done, st);
}

gbd_status fail(gbd_status code, const char *fmt, ...)
{
    va_list ap;
    va_start(ap, fmt);
    vsnprintf(g_err, sizeof g_err, fmt, ap);
    va_end(ap);
    return code;
}
gbd_status cuda_fail(cudaError_t e, const char *what)
{
    return fail(GBD_ECUDA, "%s: %s", what, cudaGetErrorString(e));
}
bool aligned16(const void *p) { return (reinterpret_cast<uintptr_t>(p) & 15u) == 0; }

// GBD_DEBUG_SYNC=1 (read once): every call that enqueued work synchronises its stream before returning and reports
// an asynchronous CUDA fault as its own error; gbd_beamlets_create additionally reads the
// lattice kernel's own count back and compares it with the host count the handle carries.
bool debug_sync_enabled()
{
    static const bool on = [] { const char *v = getenv("GBD_DEBUG_SYNC"); return v && v[0] == '1'; }();
    return on;
}
gbd_status done(cudaStream_t st, const char *what)
{
    if (!debug_sync_enabled()) return GBD_OK;
    cudaError_t e = cudaStreamSynchronize(st);
    if (e == cudaSuccess) e = cudaGetLastError();
    return e == cudaSuccess ? GBD_OK : cuda_fail(e, what);
}
size_t align_up(size_t x, size_t a) { return (x + a - 1) / a * a; }

bool detector_ok(const gbd_detector *d)
{
    if (!d || d->n_u < 1 || d->n_v < 1 || !(d->du > 0.0) || !(d->dv > 0.0)) return false;
    if (!std::isfinite(d->du) || !std::isfinite(d->dv)) return false;
    double uu = 0, vv = 0, uv = 0;
    for (int i = 0; i < 3; ++i) {
        if (!std::isfinite(d->origin[i]) || !std::isfinite(d->e_u[i]) || !std::isfinite(d->e_v[i])) return false;
        uu += d->e_u[i] * d->e_u[i];
        vv += d->e_v[i] * d->e_v[i];
        uv += d->e_u[i] * d->e_v[i];
    }
    return std::fabs(uu - 1.0) < 1e-9 && std::fabs(vv - 1.0) < 1e-9 && std::fabs(uv) < 1e-9;
}

struct EvalPlan {
    int P;
    size_t eval_bytes, partial_bytes, elem;
    GbdFieldLaunch L;
};

void make_plan(long n_b, const gbd_detector *det, int precision, int algo, EvalPlan *pl)
{
    int threads, cps;
    gbd_field_config(det->n_u, precision, algo, &pl->P, &threads, &cps);
    pl->elem = precision == GBD_PRECISION_FP64 ? 16 : 8;
    GbdFieldLaunch &L = pl->L;
    memset(&L, 0, sizeof L);
    L.n_b = n_b;
    L.geom.n_u = det->n_u; L.geom.n_v = det->n_v; L.geom.du = det->du; L.geom.dv = det->dv;
    L.geom.u0 = -0.5 * (det->n_u - 1) * det->du;
    L.geom.v0 = -0.5 * (det->n_v - 1) * det->dv;
    int warps = threads / 32;
    if (algo == GBD_ALGO_RECURRENCE) {
        // a "strip" is one thread's run of P consecutive pixels; a tile holds warps*32 of them
        L.strips_per_row = (det->n_u + pl->P - 1) / pl->P;
        L.n_strips = (long)det->n_v * L.strips_per_row;
        L.n_tiles = (L.n_strips + warps * 32 - 1) / (warps * 32);
    } else {
        int w = 32 * pl->P;
        L.strips_per_row = (det->n_u + w - 1) / w;
        L.n_strips = (long)det->n_v * L.strips_per_row;
        L.n_tiles = (L.n_strips + warps - 1) / warps;
    }
    L.tiles_per_problem = L.n_tiles;
    L.work = (long long)L.n_tiles * n_b;
    L.slots = gbd_field_slots(precision);
    // room for the recurrence records, or (algo 2) the separable records + the recurrence records of the gated
    // fallback + the gate word
    pl->eval_bytes = align_up((size_t)n_b * (GBD_NEVAL + 4) * 8, 256) + align_up((size_t)n_b * (GBD_NEVAL + 2) * 8, 256) + 256;
    // a tile is at most 8 warps x 32 lanes x 32 px of complex128 or 16 warps x 32 x 32 of complex64 (recurrence):
    // 128 KiB either way -- size for the largest so the workspace query does not depend on the algorithm
    pl->partial_bytes = align_up((size_t)L.slots * 2 * 8192 * 16, 256);
}

}  // namespace

// The same error / launch bookkeeping for entry points that live beside their kernels in another file
// (gbd_psf_metrics_static in gbd_metrics.cu); declared in gbd_common.cuh.
gbd_status gbd_api_fail(gbd_status code, const char *msg) { return fail(code, "%s", msg); }
gbd_status gbd_api_cuda_fail(cudaError_t e, const char *what) { return cuda_fail(e, what); }
gbd_status gbd_api_done(cudaStream_t st, int launches, const char *what)
{
    g_launches += launches;
    return done(st, what);
}
bool gbd_api_detector_ok(const gbd_detector *det) { return detector_ok(det); }

extern "C" {

const char *gbd_last_error(void) { return g_err; }
int gbd_record_doubles(void) { return GBD_NREC; }
long gbd_launch_count(void) { return g_launches.load(); }
void gbd_set_profile_events(void *ev_start, void *ev_stop)
{
    g_ev0 = (cudaEvent_t)ev_start;
    g_ev1 = (cudaEvent_t)ev_stop;
}

gbd_status gbd_beamlets_create(gbd_beamlets **out, int n_across, double pupil_diameter,
                               double overlap_factor, double waist, double wavelength, double *d_xy,
                               long capacity, long *n_out, void *cuda_stream)
{
    if (!out || !d_xy || !n_out) return fail(GBD_EINVAL, "gbd_beamlets_create: null pointer");
    if (n_across < 1 || n_across > 46340) return fail(GBD_EINVAL, "gbd_beamlets_create: n_across out of range");
    if (!(pupil_diameter > 0.0) || !(wavelength > 0.0))
        return fail(GBD_EINVAL, "gbd_beamlets_create: diameter and wavelength must be > 0");
    if (!(waist > 0.0) && !(overlap_factor > 0.0))
        return fail(GBD_EINVAL, "gbd_beamlets_create: need waist > 0 or overlap_factor > 0");
    if (capacity < 1 || !aligned16(d_xy)) return fail(GBD_EINVAL, "gbd_beamlets_create: bad d_xy/capacity");
    cudaStream_t st = (cudaStream_t)cuda_stream;
    double pitch = pupil_diameter / (double)n_across;
    double r2max = (0.5 * pupil_diameter) * (0.5 * pupil_diameter);
    // the count is computed on the host with the kernel's own individually rounded predicate (gbd_lattice_count,
    // bit-identical by construction and tested against the oracle), so the call does not wait for the kernel
    const long n = gbd_lattice_count(n_across, pupil_diameter);
    *n_out = n;
    if (n > capacity) return fail(GBD_ECAPACITY, "gbd_beamlets_create: %ld beamlets > capacity %ld", n, capacity);
    long *d_count = nullptr;
    if (debug_sync_enabled() && cudaMalloc(&d_count, sizeof(long)) != cudaSuccess) d_count = nullptr;
    cudaError_t e = gbd_launch_lattice(n_across, pitch, r2max, d_xy, capacity, d_count, st);
    if (e != cudaSuccess) { cudaFree(d_count); return cuda_fail(e, "lattice kernel"); }
    g_launches++;
    if (d_count) {
        long dev_n = -1;
        e = cudaMemcpyAsync(&dev_n, d_count, sizeof(long), cudaMemcpyDeviceToHost, st);
        if (e == cudaSuccess) e = cudaStreamSynchronize(st);
        cudaFree(d_count);
        if (e != cudaSuccess) return cuda_fail(e, "gbd_beamlets_create (GBD_DEBUG_SYNC)");
        if (dev_n != n)
            return fail(GBD_ESTATE, "gbd_beamlets_create: the lattice kernel kept %ld beamlets, the host predicate %ld",
                        dev_n, n);
    }
    gbd_beamlets *b = new (std::nothrow) gbd_beamlets;
    if (!b) return fail(GBD_EINVAL, "out of host memory");
    b->n = n;
    b->waist = waist > 0.0 ? waist : overlap_factor * pitch / 2.0;      // P:245 Eq. 24
    b->wavelength = wavelength;
    b->propagated = false;
    *out = b;
    return GBD_OK;
}

gbd_status gbd_beamlets_create_custom(gbd_beamlets **out, long n, double waist, double wavelength)
{
    if (!out) return fail(GBD_EINVAL, "gbd_beamlets_create_custom: null pointer");
    if (n < 0 || !(waist > 0.0) || !(wavelength > 0.0))
        return fail(GBD_EINVAL, "gbd_beamlets_create_custom: n >= 0, waist > 0, wavelength > 0 required");
    gbd_beamlets *b = new (std::nothrow) gbd_beamlets;
    if (!b) return fail(GBD_EINVAL, "out of host memory");
    b->n = n; b->waist = waist; b->wavelength = wavelength; b->propagated = false;
    *out = b;
    return GBD_OK;
}

void gbd_beamlets_destroy(gbd_beamlets *b) { delete b; }
long gbd_beamlets_count(const gbd_beamlets *b) { return b ? b->n : -1; }
double gbd_beamlets_waist(const gbd_beamlets *b) { return b ? b->waist : 0.0; }
double gbd_beamlets_wavelength(const gbd_beamlets *b) { return b ? b->wavelength : 0.0; }
size_t gbd_params_bytes(const gbd_beamlets *b) { return b ? (size_t)b->n * GBD_NREC * 8 : 0; }

gbd_status gbd_propagate_q(gbd_beamlets *b, const double *d_xy, long xy_stride, int abcd_mode,
                           const double *d_abcd, double l0, const double *d_base,
                           const double *d_weight, double *d_params, void *cuda_stream)
{
    if (!b) return fail(GBD_EINVAL, "gbd_propagate_q: null handle");
    if (abcd_mode != 0 && abcd_mode != 1) return fail(GBD_EINVAL, "gbd_propagate_q: abcd_mode must be 0 or 1");
    if (b->n == 0) { b->propagated = true; return GBD_OK; }
    if (!d_abcd || !d_params) return fail(GBD_EINVAL, "gbd_propagate_q: null d_abcd/d_params");
    if (abcd_mode == 1 && (!d_xy || xy_stride < b->n))
        return fail(GBD_EINVAL, "gbd_propagate_q: abcd_mode 1 needs d_xy with xy_stride >= n");
    if (abcd_mode == 0 && !d_base) return fail(GBD_EINVAL, "gbd_propagate_q: abcd_mode 0 needs d_base");
    if (!std::isfinite(l0)) return fail(GBD_EINVAL, "gbd_propagate_q: l0 not finite");
    if (!aligned16(d_params) || !aligned16(d_abcd)) return fail(GBD_EINVAL, "gbd_propagate_q: misaligned pointer");
    double l0_red = std::fmod(l0, b->wavelength);                         // R-9
    cudaError_t e = gbd_launch_propagate(b->n, d_xy, xy_stride, b->waist, b->wavelength, abcd_mode, d_abcd,
                                         l0_red, d_base, d_weight, d_params, (cudaStream_t)cuda_stream);
    if (e != cudaSuccess) return cuda_fail(e, "propagate kernel");
    if (b->n) g_launches++;
    b->propagated = true;
    return done((cudaStream_t)cuda_stream, "gbd_propagate_q (GBD_DEBUG_SYNC)");
}

gbd_status gbd_trace_mirrors(const gbd_beamlets *b, const double *d_xy, long xy_stride, const double *d_p_in,
                             const double *d_opl0, const gbd_trace_system *sys, double *d_abcd, double *d_base,
                             void *cuda_stream)
{
    if (!b || !sys) return fail(GBD_EINVAL, "gbd_trace_mirrors: null handle / system");
    if (b->n == 0) return GBD_OK;
    if (!d_xy || !d_abcd || !d_base || xy_stride < b->n)
        return fail(GBD_EINVAL, "gbd_trace_mirrors: null pointer or xy_stride < n");
    if (sys->n_mirrors < 0 || sys->n_mirrors > GBD_MAX_MIRRORS)
        return fail(GBD_EINVAL, "gbd_trace_mirrors: 0..%d mirrors", GBD_MAX_MIRRORS);
    if (!(sys->dq > 0.0) || !(sys->dp > 0.0) || (sys->dir_sign != 1.0 && sys->dir_sign != -1.0))
        return fail(GBD_EINVAL, "gbd_trace_mirrors: dq, dp > 0 and dir_sign = +-1 required");
    double xx = 0, yy = 0, xy = 0;
    for (int i = 0; i < 3; ++i) {
        if (!std::isfinite(sys->origin[i]) || !std::isfinite(sys->e_x[i]) || !std::isfinite(sys->e_y[i]))
            return fail(GBD_EINVAL, "gbd_trace_mirrors: evaluation frame not finite");
        xx += sys->e_x[i] * sys->e_x[i]; yy += sys->e_y[i] * sys->e_y[i]; xy += sys->e_x[i] * sys->e_y[i];
    }
    if (std::fabs(xx - 1.0) > 1e-9 || std::fabs(yy - 1.0) > 1e-9 || std::fabs(xy) > 1e-9)
        return fail(GBD_EINVAL, "gbd_trace_mirrors: e_x, e_y must be orthonormal");
    for (int m = 0; m < sys->n_mirrors; ++m)
        if (!std::isfinite(sys->mirrors[m].curvature) || !std::isfinite(sys->mirrors[m].conic) ||
            !std::isfinite(sys->mirrors[m].z_vertex))
            return fail(GBD_EINVAL, "gbd_trace_mirrors: mirror %d not finite", m);
    if (!aligned16(d_abcd)) return fail(GBD_EINVAL, "gbd_trace_mirrors: misaligned d_abcd");
    cudaError_t e = gbd_launch_trace(b->n, d_xy, xy_stride, d_p_in, d_opl0, *sys, b->wavelength, d_abcd, d_base,
                                     (cudaStream_t)cuda_stream);
    if (e != cudaSuccess) return cuda_fail(e, "trace kernel");
    g_launches++;
    return done((cudaStream_t)cuda_stream, "gbd_trace_mirrors (GBD_DEBUG_SYNC)");
}

size_t gbd_eval_workspace_bytes(const gbd_beamlets *b, const gbd_detector *det, int precision)
{
    if (!b || !detector_ok(det)) return 0;
    EvalPlan pl;
    make_plan(b->n, det, precision, GBD_ALGO_DIRECT, &pl);
    return pl.eval_bytes + pl.partial_bytes;
}

gbd_status gbd_eval_field(const gbd_beamlets *b, const double *d_params, const gbd_detector *det,
                          int precision, int algo, double cull_tau, void *d_field, void *d_workspace,
                          size_t workspace_bytes, void *cuda_stream)
{
    if (!b || !d_field || !d_workspace || (!d_params && b->n > 0))
        return fail(GBD_EINVAL, "gbd_eval_field: null pointer");
    if (!b->propagated) return fail(GBD_ESTATE, "gbd_eval_field: call gbd_propagate_q first");
    if (!detector_ok(det)) return fail(GBD_EINVAL, "gbd_eval_field: bad detector (sizes > 0, axes orthonormal)");
    if (precision != GBD_PRECISION_FP64 && precision != GBD_PRECISION_MIXED)
        return fail(GBD_EINVAL, "gbd_eval_field: precision must be 0 or 1");
    if (algo != GBD_ALGO_DIRECT && algo != GBD_ALGO_RECURRENCE && algo != GBD_ALGO_SEPARABLE)
        return fail(GBD_EINVAL, "gbd_eval_field: algo must be 0, 1 or 2");
    if (algo != GBD_ALGO_DIRECT && cull_tau > 0.0)
        return fail(GBD_EINVAL, "gbd_eval_field: only algo 0 has a cull");
    if (!aligned16(d_field) || (reinterpret_cast<uintptr_t>(d_workspace) & 127u) || !aligned16(d_params))
        return fail(GBD_EINVAL, "gbd_eval_field: misaligned pointer (field/params 16 B, workspace 128 B)");
    if (std::isnan(cull_tau)) return fail(GBD_EINVAL, "gbd_eval_field: cull_tau is NaN");
    cudaStream_t st = (cudaStream_t)cuda_stream;
    if (algo != GBD_ALGO_DIRECT && det->n_u < 16) algo = GBD_ALGO_DIRECT;        // rows too short to pay
    const bool separable = algo == GBD_ALGO_SEPARABLE;
    if (separable) algo = GBD_ALGO_RECURRENCE;                                   // plan of the gated fallback
    EvalPlan pl;
    make_plan(b->n, det, precision, algo, &pl);
    if (workspace_bytes < pl.eval_bytes + pl.partial_bytes)
        return fail(GBD_ECAPACITY, "gbd_eval_field: workspace %zu < %zu bytes", workspace_bytes,
                    pl.eval_bytes + pl.partial_bytes);
    size_t field_bytes = (size_t)det->n_u * det->n_v * pl.elem;
    if (b->n == 0) {
        cudaError_t e = cudaMemsetAsync(d_field, 0, field_bytes, st);
        return e == cudaSuccess ? GBD_OK : cuda_fail(e, "memset");
    }
    double *d_eval = reinterpret_cast<double *>(d_workspace);
    pl.L.rec = d_eval;
    pl.L.out = d_field;
    pl.L.partial = reinterpret_cast<char *>(d_workspace) + pl.eval_bytes;
    const bool cull = cull_tau > 0.0;
    pl.L.log2_tau = cull ? std::log2(cull_tau) : 0.0;
    if (separable) {
        // workspace: [separable records][recurrence records][gate]; the pre-pass raises the gate when a beamlet
        // has a cross term; the separable kernels run on gate == 0, the recurrence kernels on gate == 1
        char *base = reinterpret_cast<char *>(d_workspace);
        double *d_ev16 = d_eval;
        double *d_ev14 = reinterpret_cast<double *>(base + align_up((size_t)b->n * (GBD_NEVAL + 4) * 8, 256));
        int *d_gate = reinterpret_cast<int *>(base + pl.eval_bytes - 256);
        cudaError_t e = cudaMemsetAsync(d_gate, 0, sizeof(int), st);
        if (e == cudaSuccess)
            e = gbd_launch_prepass(b->n, d_params, *det, b->wavelength, GBD_PRECISION_FP64, GBD_ALGO_SEPARABLE,
                                   d_ev16, d_gate, st);
        if (e == cudaSuccess)
            e = gbd_launch_prepass(b->n, d_params, *det, b->wavelength, GBD_PRECISION_FP64, GBD_ALGO_RECURRENCE,
                                   d_ev14, nullptr, st);
        if (e != cudaSuccess) return cuda_fail(e, "pre-pass kernels");
        g_launches += 2;
        GbdFieldLaunch Ls = pl.L;
        int tiles_u = 0;
        gbd_sep_geometry(det->n_u, det->n_v, precision, &tiles_u, &Ls.n_tiles);
        Ls.strips_per_row = tiles_u;
        Ls.n_strips = Ls.n_tiles;
        Ls.tiles_per_problem = Ls.n_tiles;
        Ls.work = (long long)Ls.n_tiles * b->n;
        Ls.rec = d_ev16;
        Ls.gate = d_gate;
        Ls.gate_want = 0;
        Ls.slots = gbd_sep_slots(precision, pl.L.slots);
        int nl = 0;
        e = gbd_launch_field_sep(Ls, precision, &nl, st, g_ev0, g_ev1);
        if (e != cudaSuccess) return cuda_fail(e, "separable field-sum kernel");
        g_launches += nl;
        pl.L.rec = d_ev14;
        pl.L.gate = d_gate;
        pl.L.gate_want = 1;
        e = gbd_launch_field(pl.L, pl.P, precision, GBD_ALGO_RECURRENCE, false, &nl, st, nullptr, nullptr);
        if (e != cudaSuccess) return cuda_fail(e, "gated recurrence field-sum kernel");
        g_launches += nl;
        return done(st, "gbd_eval_field (GBD_DEBUG_SYNC)");
    }
    // table kernels: the pre-pass tells them on the device whether any envelope exponent leaves [-1000, 1000]
    int *d_deep = nullptr;
    double *d_eval_abs = nullptr;
    cudaError_t e = cudaSuccess;
    if (gbd_field_uses_tables(pl.L, pl.P, precision, algo)) {
        d_deep = reinterpret_cast<int *>(reinterpret_cast<char *>(d_workspace) + pl.eval_bytes - 256) + 1;
        e = cudaMemsetAsync(d_deep, 0, sizeof(int), st);
        if (e != cudaSuccess) return cuda_fail(e, "memset");
        pl.L.deep = d_deep;
        // the plain table kernel also gets the records in detector coordinates (second record region of the workspace)
        if (!cull)
            d_eval_abs = reinterpret_cast<double *>(reinterpret_cast<char *>(d_workspace) +
                                                    align_up((size_t)b->n * (GBD_NEVAL + 4) * 8, 256));
        pl.L.rec_abs = d_eval_abs;
    }
    // the recurrence kernels (either precision) read the fp64 record layout + S
    e = gbd_launch_prepass(b->n, d_params, *det, b->wavelength,
                           algo == GBD_ALGO_RECURRENCE ? GBD_PRECISION_FP64 : precision, algo, d_eval, nullptr, st,
                           d_deep, d_eval_abs);
    if (e != cudaSuccess) return cuda_fail(e, "pre-pass kernel");
    g_launches++;
    int nl = 0;
    e = gbd_launch_field(pl.L, pl.P, precision, algo, cull, &nl, st, g_ev0, g_ev1);
    if (e != cudaSuccess) return cuda_fail(e, "field-sum kernel");
    g_launches += nl;
    return done(st, "gbd_eval_field (GBD_DEBUG_SYNC)");
}

size_t gbd_host_workspace_bytes(const gbd_beamlets *b, const gbd_detector *det, int abcd_mode, int precision)
{
    if (!b || !detector_ok(det)) return 0;
    size_t n = (size_t)b->n;
    size_t s = 0;
    s += align_up(2 * n * 8, 256);                                 // xy
    s += align_up((abcd_mode ? 16 : 16 * n) * 8, 256);             // abcd
    s += align_up(5 * n * 8, 256);                                 // base
    s += align_up(2 * n * 8, 256);                                 // weight
    s += align_up(n * GBD_NREC * 8, 256);                          // params
    s += align_up((size_t)det->n_u * det->n_v * (precision ? 8 : 16), 256);   // field
    s += gbd_eval_workspace_bytes(b, det, precision);
    return s;
}

gbd_status gbd_eval_field_host(gbd_beamlets *b, const double *h_xy, int abcd_mode, const double *h_abcd,
                               double l0, const double *h_base, const double *h_weight,
                               const gbd_detector *det, int precision, int algo, double cull_tau,
                               void *h_field, void *d_workspace, size_t workspace_bytes, void *cuda_stream)
{
    if (!b || !h_abcd || !h_field || !d_workspace) return fail(GBD_EINVAL, "gbd_eval_field_host: null pointer");
    if (abcd_mode != 0 && abcd_mode != 1) return fail(GBD_EINVAL, "gbd_eval_field_host: abcd_mode must be 0 or 1");
    if (abcd_mode == 1 && !h_xy) return fail(GBD_EINVAL, "gbd_eval_field_host: abcd_mode 1 needs h_xy");
    if (abcd_mode == 0 && !h_base) return fail(GBD_EINVAL, "gbd_eval_field_host: abcd_mode 0 needs h_base");
    if (!detector_ok(det)) return fail(GBD_EINVAL, "gbd_eval_field_host: bad detector");
    if (reinterpret_cast<uintptr_t>(d_workspace) & 255u) return fail(GBD_EINVAL, "gbd_eval_field_host: workspace must be 256-byte aligned");
    size_t need = gbd_host_workspace_bytes(b, det, abcd_mode, precision);
    if (workspace_bytes < need)
        return fail(GBD_ECAPACITY, "gbd_eval_field_host: workspace %zu < %zu bytes", workspace_bytes, need);
    cudaStream_t st = (cudaStream_t)cuda_stream;
    size_t n = (size_t)b->n;
    char *p = reinterpret_cast<char *>(d_workspace);
    auto carve = [&](size_t bytes) { char *q = p; p += align_up(bytes, 256); return q; };
    double *d_xy = (double *)carve(2 * n * 8);
    double *d_abcd = (double *)carve((abcd_mode ? 16 : 16 * n) * 8);
    double *d_base = (double *)carve(5 * n * 8);
    double *d_weight = (double *)carve(2 * n * 8);
    double *d_params = (double *)carve(n * GBD_NREC * 8);
    size_t field_bytes = (size_t)det->n_u * det->n_v * (precision ? 8 : 16);
    void *d_field = carve(field_bytes);
    size_t ws_left = workspace_bytes - (size_t)(p - reinterpret_cast<char *>(d_workspace));
    cudaError_t e = cudaSuccess;
    auto h2d = [&](void *d, const void *h, size_t bytes) {
        if (e == cudaSuccess && h && bytes) e = cudaMemcpyAsync(d, h, bytes, cudaMemcpyHostToDevice, st);
    };
    h2d(d_xy, h_xy, 2 * n * 8);
    h2d(d_abcd, h_abcd, (abcd_mode ? 16 : 16 * n) * 8);
    h2d(d_base, h_base, (abcd_mode ? 3 : 5) * n * 8);
    h2d(d_weight, h_weight, 2 * n * 8);
    if (e != cudaSuccess) return cuda_fail(e, "H2D copy");
    gbd_status s = gbd_propagate_q(b, d_xy, (long)n, abcd_mode, d_abcd, l0, h_base ? d_base : nullptr,
                                   h_weight ? d_weight : nullptr, d_params, cuda_stream);
    if (s != GBD_OK) return s;
    s = gbd_eval_field(b, d_params, det, precision, algo, cull_tau, d_field, p, ws_left, cuda_stream);
    if (s != GBD_OK) return s;
    e = cudaMemcpyAsync(h_field, d_field, field_bytes, cudaMemcpyDeviceToHost, st);
    if (e == cudaSuccess) e = cudaStreamSynchronize(st);
    if (e != cudaSuccess) return cuda_fail(e, "D2H copy / synchronise");
    return GBD_OK;
}

gbd_status gbd_probe_dfma(double *d_sink, long iters, double *dfma_per_launch, void *cuda_stream)
{
    if (!d_sink || iters < 1) return fail(GBD_EINVAL, "gbd_probe_dfma: bad arguments");
    cudaError_t e = gbd_launch_probe(d_sink, iters, dfma_per_launch, (cudaStream_t)cuda_stream);
    if (e != cudaSuccess) return cuda_fail(e, "probe kernel");
    g_launches++;
    return GBD_OK;
}

static bool detector_untilted(const gbd_detector *d)
{
    return d->e_u[0] == 1.0 && d->e_u[1] == 0.0 && d->e_u[2] == 0.0 && d->e_v[0] == 0.0 && d->e_v[1] == 1.0 &&
           d->e_v[2] == 0.0 && d->origin[2] == 0.0;
}

gbd_status gbd_hg_modes(const gbd_beamlets *b, int abcd_mode, const double *d_abcd, const double *d_mode_weight,
                        double *d_modes, void *cuda_stream)
{
    if (!b || !d_abcd || (!d_modes && b->n > 0)) return fail(GBD_EINVAL, "gbd_hg_modes: null pointer");
    if (abcd_mode != 0 && abcd_mode != 1) return fail(GBD_EINVAL, "gbd_hg_modes: abcd_mode must be 0 or 1");
    if (!aligned16(d_abcd) || !aligned16(d_modes) || !aligned16(d_mode_weight))
        return fail(GBD_EINVAL, "gbd_hg_modes: misaligned pointer (16 B)");
    cudaError_t e = gbd_launch_hg_modes(b->n, b->waist, b->wavelength, abcd_mode, d_abcd, d_mode_weight, d_modes,
                                        (cudaStream_t)cuda_stream);
    if (e != cudaSuccess) return cuda_fail(e, "mode-factor kernel");
    if (b->n > 0) g_launches++;
    return done((cudaStream_t)cuda_stream, "gbd_hg_modes (GBD_DEBUG_SYNC)");
}

size_t gbd_eval_modes_workspace_bytes(const gbd_beamlets *b, const gbd_detector *det)
{
    if (!b || !detector_ok(det)) return 0;
    EvalPlan pl;
    make_plan(b->n, det, GBD_PRECISION_FP64, GBD_ALGO_DIRECT, &pl);
    // [beamlet-centred records][gate words][detector-coordinate records][stream-K partials]
    return 2 * align_up((size_t)b->n * GBD_NEVAL_HG * 8, 256) + 256 + pl.partial_bytes;
}

gbd_status gbd_eval_field_modes(const gbd_beamlets *b, const double *d_params, const double *d_modes,
                                const gbd_detector *det, void *d_field, void *d_workspace, size_t workspace_bytes,
                                void *cuda_stream)
{
    if (!b || !d_field || !d_workspace || ((!d_params || !d_modes) && b->n > 0))
        return fail(GBD_EINVAL, "gbd_eval_field_modes: null pointer");
    if (!b->propagated) return fail(GBD_ESTATE, "gbd_eval_field_modes: call gbd_propagate_q first");
    if (!detector_ok(det)) return fail(GBD_EINVAL, "gbd_eval_field_modes: bad detector (sizes > 0, axes orthonormal)");
    if (!detector_untilted(det))
        return fail(GBD_EINVAL, "gbd_eval_field_modes: the detector must be untilted (e_u = X, e_v = Y, origin z = 0)");
    if (!aligned16(d_field) || (reinterpret_cast<uintptr_t>(d_workspace) & 127u) || !aligned16(d_params) ||
        !aligned16(d_modes))
        return fail(GBD_EINVAL, "gbd_eval_field_modes: misaligned pointer (field/params/modes 16 B, workspace 128 B)");
    const size_t need = gbd_eval_modes_workspace_bytes(b, det);
    if (workspace_bytes < need)
        return fail(GBD_ECAPACITY, "gbd_eval_field_modes: workspace %zu < %zu bytes", workspace_bytes, need);
    cudaStream_t st = (cudaStream_t)cuda_stream;
    if (b->n == 0) {
        cudaError_t e = cudaMemsetAsync(d_field, 0, (size_t)det->n_u * det->n_v * 16, st);
        return e == cudaSuccess ? GBD_OK : cuda_fail(e, "memset");
    }
    EvalPlan pl;
    make_plan(b->n, det, GBD_PRECISION_FP64, GBD_ALGO_DIRECT, &pl);
    double *d_eval = reinterpret_cast<double *>(d_workspace);
    pl.L.rec = d_eval;
    pl.L.out = d_field;
    const size_t rec_bytes = align_up((size_t)b->n * GBD_NEVAL_HG * 8, 256);
    pl.L.partial = reinterpret_cast<char *>(d_workspace) + 2 * rec_bytes + 256;
    int *d_deep = nullptr;
    double *d_eval_abs = nullptr;
    cudaError_t e = cudaSuccess;
    if (gbd_field_uses_tables(pl.L, pl.P, GBD_PRECISION_FP64, GBD_ALGO_DIRECT)) {
        // last 256 bytes of the record area (its size is rounded up and padded in gbd_eval_modes_workspace_bytes)
        d_deep = reinterpret_cast<int *>(reinterpret_cast<char *>(d_workspace) + align_up((size_t)b->n * GBD_NEVAL_HG * 8, 256));
        e = cudaMemsetAsync(d_deep, 0, sizeof(int), st);
        if (e != cudaSuccess) return cuda_fail(e, "memset");
        pl.L.deep = d_deep;
        d_eval_abs = reinterpret_cast<double *>(reinterpret_cast<char *>(d_workspace) + rec_bytes + 256);
        pl.L.rec_abs = d_eval_abs;
    }
    e = gbd_launch_prepass_modes(b->n, d_params, d_modes, *det, b->wavelength, d_eval, st, d_deep, d_eval_abs);
    if (e != cudaSuccess) return cuda_fail(e, "mode pre-pass kernel");
    g_launches++;
    int nl = 0;
    e = gbd_launch_field_modes(pl.L, pl.P, &nl, st, g_ev0, g_ev1);
    if (e != cudaSuccess) return cuda_fail(e, "mode field-sum kernel");
    g_launches += nl;
    return done(st, "gbd_eval_field_modes (GBD_DEBUG_SYNC)");
}

size_t gbd_pointeval_workspace_bytes(const gbd_beamlets *b, const gbd_detector *det)
{
    if (!b || !detector_ok(det)) return 0;
    const long n_px = (long)det->n_u * det->n_v;
    const int splits = gbd_pointeval_splits(b->n, n_px, gbd_field_slots(GBD_PRECISION_FP64));
    return align_up(gbd_pointeval_record_bytes(b->n), 256) + (splits > 1 ? (size_t)splits * n_px * 16 : 0) + 256;
}

gbd_status gbd_eval_field_pointwise(const gbd_beamlets *b, const double *d_xy, long xy_stride, int abcd_mode,
                                    const double *d_abcd, double l0, const double *d_base, const double *d_weight,
                                    const gbd_detector *det, void *d_field, void *d_workspace,
                                    size_t workspace_bytes, void *cuda_stream)
{
    if (!b || !d_abcd || !d_field || !d_workspace) return fail(GBD_EINVAL, "gbd_eval_field_pointwise: null pointer");
    if (abcd_mode != 0 && abcd_mode != 1) return fail(GBD_EINVAL, "gbd_eval_field_pointwise: abcd_mode must be 0 or 1");
    if (abcd_mode == 0 && !d_base && b->n > 0)
        return fail(GBD_EINVAL, "gbd_eval_field_pointwise: abcd_mode 0 needs d_base");
    if (abcd_mode == 1 && (!d_xy || xy_stride < b->n) && b->n > 0)
        return fail(GBD_EINVAL, "gbd_eval_field_pointwise: abcd_mode 1 needs d_xy with xy_stride >= n");
    if (!detector_ok(det)) return fail(GBD_EINVAL, "gbd_eval_field_pointwise: bad detector (sizes > 0, axes orthonormal)");
    if (!std::isfinite(l0)) return fail(GBD_EINVAL, "gbd_eval_field_pointwise: l0 is not finite");
    if (!aligned16(d_field) || !aligned16(d_abcd) || (reinterpret_cast<uintptr_t>(d_workspace) & 255u))
        return fail(GBD_EINVAL, "gbd_eval_field_pointwise: misaligned pointer (field/abcd 16 B, workspace 256 B)");
    const size_t need = gbd_pointeval_workspace_bytes(b, det);
    if (workspace_bytes < need)
        return fail(GBD_ECAPACITY, "gbd_eval_field_pointwise: workspace %zu < %zu bytes", workspace_bytes, need);
    cudaStream_t st = (cudaStream_t)cuda_stream;
    const long n_px = (long)det->n_u * det->n_v;
    if (b->n == 0) {
        cudaError_t e = cudaMemsetAsync(d_field, 0, (size_t)n_px * 16, st);
        return e == cudaSuccess ? GBD_OK : cuda_fail(e, "memset");
    }
    const int splits = gbd_pointeval_splits(b->n, n_px, gbd_field_slots(GBD_PRECISION_FP64));
    char *base = reinterpret_cast<char *>(d_workspace);
    double *d_rec = reinterpret_cast<double *>(base);
    void *d_part = base + align_up(gbd_pointeval_record_bytes(b->n), 256);
    int nl = 0;
    cudaError_t e = gbd_launch_pointeval(b->n, d_xy, xy_stride, b->waist, b->wavelength, abcd_mode, d_abcd,
                                         std::fmod(l0, b->wavelength), d_base, d_weight, *det, splits, d_rec, d_part,
                                         d_field, &nl, st, g_ev0, g_ev1);
    if (e != cudaSuccess) return cuda_fail(e, "point-evaluation kernels");
    g_launches += nl;
    return done(st, "gbd_eval_field_pointwise (GBD_DEBUG_SYNC)");
}

size_t gbd_psf_metrics_workspace_bytes(const gbd_detector *det)
{
    if (!detector_ok(det)) return 0;
    return align_up((size_t)gbd_metrics_blocks((long)det->n_u * det->n_v) * 9 * 8, 256);
}

gbd_status gbd_psf_metrics(const void *d_field, int precision, const gbd_detector *det, double lambda_fnum,
                           const double *d_e0, double *d_metrics, void *d_workspace, size_t workspace_bytes,
                           void *cuda_stream)
{
    if (!d_field || !d_e0 || !d_metrics || !d_workspace) return fail(GBD_EINVAL, "gbd_psf_metrics: null pointer");
    if (!detector_ok(det)) return fail(GBD_EINVAL, "gbd_psf_metrics: bad detector");
    if (precision != 0 && precision != 1) return fail(GBD_EINVAL, "gbd_psf_metrics: precision must be 0 or 1");
    if (!(lambda_fnum > 0.0)) return fail(GBD_EINVAL, "gbd_psf_metrics: lambda_fnum must be > 0");
    if (workspace_bytes < gbd_psf_metrics_workspace_bytes(det))
        return fail(GBD_ECAPACITY, "gbd_psf_metrics: workspace too small");
    cudaError_t e = gbd_launch_metrics(d_field, precision, *det, lambda_fnum, d_e0, d_metrics,
                                       (double *)d_workspace, 1, 9, nullptr, (cudaStream_t)cuda_stream);
    if (e != cudaSuccess) return cuda_fail(e, "metrics kernels");
    g_launches += 2;
    return done((cudaStream_t)cuda_stream, "gbd_psf_metrics (GBD_DEBUG_SYNC)");
}

long gbd_lattice_count(int n_across, double pupil_diameter)
{
    if (n_across < 1 || n_across > 46340 || !(pupil_diameter > 0.0)) return -1;
    const double pitch = pupil_diameter / (double)n_across;
    const double r2max = (0.5 * pupil_diameter) * (0.5 * pupil_diameter);
    const double half = 0.5 * (double)(n_across - 1);
    // the kernel's predicate, every product and the sum individually rounded (volatile: no contraction)
    auto keep = [&](int ix, double yy) {
        volatile double x = ((double)ix - half) * pitch;
        volatile double xx = x * x;
        volatile double r2 = xx + yy;
        return r2 <= r2max;
    };
    // rounding is monotone, so along a row the predicate is monotone in |ix - half| and symmetric about the
    // centre: bisect for the first kept index of the left half; the row keeps n_across - 2 * first
    const int mid = (n_across + 1) / 2;              // left half incl. the centre column of an odd lattice
    long n = 0;
    for (int iy = 0; iy < n_across; ++iy) {
        volatile double y = ((double)iy - half) * pitch;
        volatile double yy = y * y;
        int lo = 0, hi = mid;                        // first kept index in [0, mid], mid = none
        while (lo < hi) {
            const int m = (lo + hi) / 2;
            if (keep(m, yy)) hi = m; else lo = m + 1;
        }
        if (lo < mid) n += n_across - 2 * lo;
    }
    return n;
}

namespace {
struct SweepPlan {
    EvalPlan pl;
    int algo, rec_stride;
    bool separable;          // algo 2: separable kernels gated on, plan `pl` (recurrence) gated off
    size_t n_px, total_b;
    // workspace offsets
    size_t off_xy, off_params, off_eval, off_eval16, off_fields, off_e0, off_counts, off_probs, off_probs16, off_gate,
        off_jobs, off_mpart, off_partial, total;
};

bool sweep_plan(const gbd_sweep_run *runs, int n_runs, const gbd_detector *det, int precision, int algo,
                bool with_fields, SweepPlan *sp)
{
    if (!runs || n_runs < 1 || n_runs > 65535 || !detector_ok(det)) return false;
    size_t total_b = 0;
    for (int r = 0; r < n_runs; ++r) {
        long n = gbd_lattice_count(runs[r].n_across, runs[r].pupil_diameter);
        if (n < 1 || !(runs[r].wavelength > 0.0) || !(runs[r].overlap_factor > 0.0)) return false;
        total_b += (size_t)n;
    }
    if (algo != GBD_ALGO_DIRECT && det->n_u < 16) algo = GBD_ALGO_DIRECT;
    sp->separable = algo == GBD_ALGO_SEPARABLE;
    if (sp->separable) algo = GBD_ALGO_RECURRENCE;
    sp->algo = algo;
    make_plan(1, det, precision, algo, &sp->pl);
    sp->rec_stride = algo == GBD_ALGO_RECURRENCE ? GBD_NEVAL + 2 : GBD_NEVAL;
    sp->n_px = (size_t)det->n_u * det->n_v;
    sp->total_b = total_b;
    size_t o = 0;
    auto carve = [&](size_t bytes) { size_t q = o; o += align_up(bytes, 256); return q; };
    sp->off_xy = carve((2 * total_b + 2 * (size_t)n_runs * 32) * 8);     // each run's slice 256-byte aligned
    sp->off_params = carve(total_b * GBD_NREC * 8 + (size_t)n_runs * 256);
    sp->off_eval = carve(total_b * (GBD_NEVAL + 2) * 8 + (size_t)n_runs * 256);
    sp->off_eval16 = carve(total_b * (GBD_NEVAL + 4) * 8 + (size_t)n_runs * 256);
    sp->off_probs16 = carve((size_t)n_runs * sizeof(GbdProblem));
    sp->off_gate = carve(256);
    sp->off_jobs = carve((size_t)n_runs * sizeof(GbdRunJob));
    sp->off_fields = carve(with_fields ? sp->n_px * sp->pl.elem * (size_t)n_runs : 0);
    sp->off_e0 = carve((size_t)n_runs * 2 * 8);
    sp->off_counts = carve((size_t)n_runs * sizeof(long));
    sp->off_probs = carve((size_t)n_runs * sizeof(GbdProblem));
    sp->off_mpart = carve((size_t)n_runs * gbd_metrics_blocks((long)sp->n_px) * 9 * 8);
    sp->off_partial = carve(sp->pl.partial_bytes);
    sp->total = o;
    return true;
}
}  // namespace

size_t gbd_airy_sweep_workspace_bytes(const gbd_sweep_run *h_runs, int n_runs, const gbd_detector *det,
                                      int precision, int with_fields)
{
    SweepPlan sp;
    if (!sweep_plan(h_runs, n_runs, det, precision, GBD_ALGO_RECURRENCE, with_fields != 0, &sp)) return 0;
    return sp.total;
}

gbd_status gbd_airy_sweep(const gbd_sweep_run *h_runs, int n_runs, const double *d_abcd, double l0,
                          const gbd_detector *det, double lambda_fnum, int precision, int algo,
                          double *d_metrics, void *d_fields, void *d_workspace, size_t workspace_bytes,
                          void *cuda_stream)
{
    if (!h_runs || !d_abcd || !d_metrics || !d_workspace) return fail(GBD_EINVAL, "gbd_airy_sweep: null pointer");
    if (precision != GBD_PRECISION_FP64 && precision != GBD_PRECISION_MIXED)
        return fail(GBD_EINVAL, "gbd_airy_sweep: precision must be 0 or 1");
    if (algo != GBD_ALGO_DIRECT && algo != GBD_ALGO_RECURRENCE && algo != GBD_ALGO_SEPARABLE)
        return fail(GBD_EINVAL, "gbd_airy_sweep: algo must be 0, 1 or 2");
    if (!(lambda_fnum > 0.0) || !std::isfinite(l0)) return fail(GBD_EINVAL, "gbd_airy_sweep: bad lambda_fnum / l0");
    if ((reinterpret_cast<uintptr_t>(d_workspace) & 255u) || !aligned16(d_abcd) || !aligned16(d_metrics) ||
        (d_fields && !aligned16(d_fields)))
        return fail(GBD_EINVAL, "gbd_airy_sweep: misaligned pointer (workspace 256 B, others 16 B)");
    {
        // the host tables of this call go up through a process-wide pinned staging buffer (and the first call
        // allocates it): neither is capturable, and a captured copy would replay stale tables
        cudaStreamCaptureStatus cs = cudaStreamCaptureStatusNone;
        if (cudaStreamIsCapturing((cudaStream_t)cuda_stream, &cs) == cudaSuccess && cs != cudaStreamCaptureStatusNone)
            return fail(GBD_ESTATE, "gbd_airy_sweep: the stream is capturing; this call cannot be captured into a CUDA graph");
    }
    SweepPlan sp;
    if (!sweep_plan(h_runs, n_runs, det, precision, algo, d_fields == nullptr, &sp))
        return fail(GBD_EINVAL, "gbd_airy_sweep: bad runs (1..65535 runs, n_across >= 1, sizes > 0) or detector");
    if (workspace_bytes < sp.total)
        return fail(GBD_ECAPACITY, "gbd_airy_sweep: workspace %zu < %zu bytes", workspace_bytes, sp.total);
    cudaStream_t st = (cudaStream_t)cuda_stream;
    char *base = reinterpret_cast<char *>(d_workspace);
    char *fields = d_fields ? reinterpret_cast<char *>(d_fields) : base + sp.off_fields;
    long *d_counts = reinterpret_cast<long *>(base + sp.off_counts);
    GbdProblem *d_probs = reinterpret_cast<GbdProblem *>(base + sp.off_probs);
    std::vector<GbdProblem> probs((size_t)n_runs), probs16(sp.separable ? (size_t)n_runs : 0);
    GbdFieldLaunch &L = sp.pl.L;
    const long tpp = L.n_tiles;                      // tiles per problem (same detector for every run)
    long long work = 0, work16 = 0;
    size_t o_xy = 0, o_par = 0, o_ev = 0, o_ev16 = 0;
    cudaError_t e = cudaSuccess;
    long launches = 0;
    int tiles_u16 = 0;
    long tpp16 = 0;
    int *d_gate = reinterpret_cast<int *>(base + sp.off_gate);
    if (sp.separable) {
        gbd_sep_geometry(det->n_u, det->n_v, precision, &tiles_u16, &tpp16);
        e = cudaMemsetAsync(d_gate, 0, sizeof(int), st);
    }
    std::vector<GbdRunJob> jobs((size_t)n_runs);
    long max_n = 0;
    for (int r = 0; r < n_runs; ++r) {
        const gbd_sweep_run &R = h_runs[r];
        const long n = gbd_lattice_count(R.n_across, R.pupil_diameter);
        const double pitch = R.pupil_diameter / (double)R.n_across;
        const double w0 = R.overlap_factor * pitch / 2.0;                 // P:245 Eq. 24
        GbdRunJob &J = jobs[r];
        J.n_across = R.n_across;
        J.n = n;
        J.pitch = pitch;
        J.r2max = (0.5 * R.pupil_diameter) * (0.5 * R.pupil_diameter);
        J.xy = reinterpret_cast<double *>(base + sp.off_xy + o_xy);
        J.count = d_counts + r;
        J.q1_im = -R.wavelength / (3.14159265358979323846 * w0 * w0);
        J.lambda = R.wavelength;
        J.l0_red = std::fmod(l0, R.wavelength);
        J.params = reinterpret_cast<double *>(base + sp.off_params + o_par);
        J.ev = reinterpret_cast<double *>(base + sp.off_eval + o_ev);
        J.ev2 = nullptr;
        o_xy += align_up(2 * (size_t)n * 8, 256);
        o_par += align_up((size_t)n * GBD_NREC * 8, 256);
        o_ev += align_up((size_t)n * sp.rec_stride * 8, 256);
        if (n > max_n) max_n = n;
        if (sp.separable) {
            J.ev2 = reinterpret_cast<double *>(base + sp.off_eval16 + o_ev16);
            o_ev16 += align_up((size_t)n * (GBD_NEVAL + 4) * 8, 256);
            probs16[r].rec = J.ev2;
            probs16[r].out = fields + (size_t)r * sp.n_px * sp.pl.elem;
            probs16[r].n_b = n;
            probs16[r].work_begin = work16;
            work16 += (long long)tpp16 * n;
        }
        probs[r].rec = J.ev;
        probs[r].out = fields + (size_t)r * sp.n_px * sp.pl.elem;
        probs[r].n_b = n;
        probs[r].work_begin = work;
        work += (long long)tpp * n;
    }
    // direct fp64 sweeps on the table kernels: every run also gets its records in detector coordinates (they live in
    // the region the separable layout would use)
    bool sweep_tables = false;
    {
        GbdFieldLaunch Lw = L;
        Lw.work = work;
        sweep_tables = !sp.separable && gbd_field_uses_tables(Lw, sp.pl.P, precision, sp.algo);
    }
    if (sweep_tables) {
        size_t o_abs = 0;
        for (int r = 0; r < n_runs; ++r) {
            jobs[r].ev2 = reinterpret_cast<double *>(base + sp.off_eval16 + o_abs);
            probs[r].rec_abs = jobs[r].ev2;
            o_abs += align_up((size_t)jobs[r].n * (GBD_NEVAL + 4) * 8, 256);
        }
    }
    // the three host tables go up through the pinned staging buffer (no host wait on the stream)
    GbdRunJob *d_jobs = reinterpret_cast<GbdRunJob *>(base + sp.off_jobs);
    GbdProblem *d_probs16 = reinterpret_cast<GbdProblem *>(base + sp.off_probs16);
    if (e == cudaSuccess) {
        Upload up[3] = { { d_jobs, jobs.data(), (size_t)n_runs * sizeof(GbdRunJob) },
                         { d_probs, probs.data(), (size_t)n_runs * sizeof(GbdProblem) },
                         { d_probs16, probs16.data(), probs16.size() * sizeof(GbdProblem) } };
        e = staged_upload(up, sp.separable ? 3 : 2, st);
    }
    // table kernels (direct fp64 sweeps): the pre-passes report whether any envelope exponent leaves [-1000, 1000]
    int *d_deep = nullptr;
    if (sweep_tables && e == cudaSuccess) {
        d_deep = d_gate + 1;
        e = cudaMemsetAsync(d_deep, 0, sizeof(int), st);
    }
    // lattice, parameters and pre-pass of ALL runs: one launch each (grid.y = run)
    if (e == cudaSuccess) {
        int ns = 0;
        e = gbd_launch_sweep_setup(d_jobs, n_runs, max_n, d_abcd, *det, precision, sp.algo, sp.separable, d_gate, &ns, st,
                                   d_deep);
        launches += ns;
    }
    if (e != cudaSuccess) return cuda_fail(e, "gbd_airy_sweep: table upload / per-run kernels");
    L.rec = nullptr; L.n_b = 0; L.out = nullptr;
    L.probs = d_probs; L.n_probs = n_runs;
    L.tiles_per_problem = tpp;
    L.n_tiles = tpp * n_runs;
    L.work = work;
    L.partial = base + sp.off_partial;
    L.log2_tau = 0.0;
    L.deep = d_deep;
    int nl = 0;
    if (sp.separable) {
        // separable kernels run when no beamlet of any run has a cross term (gate 0), else the recurrence kernels
        GbdFieldLaunch Ls = L;
        Ls.probs = d_probs16;
        Ls.strips_per_row = tiles_u16;
        Ls.tiles_per_problem = tpp16;
        Ls.n_tiles = tpp16 * n_runs;
        Ls.n_strips = Ls.n_tiles;
        Ls.work = work16;
        Ls.gate = d_gate;
        Ls.gate_want = 0;
        Ls.slots = gbd_sep_slots(precision, L.slots);
        e = gbd_launch_field_sep(Ls, precision, &nl, st, g_ev0, g_ev1);
        if (e != cudaSuccess) return cuda_fail(e, "gbd_airy_sweep: separable field-sum kernel");
        launches += nl;
        L.gate = d_gate;
        L.gate_want = 1;
    }
    e = gbd_launch_field(L, sp.pl.P, precision, sp.algo, false, &nl, st, sp.separable ? nullptr : g_ev0,
                         sp.separable ? nullptr : g_ev1);
    if (e != cudaSuccess) return cuda_fail(e, "gbd_airy_sweep: field-sum kernel");
    launches += nl;
    double *d_e0 = reinterpret_cast<double *>(base + sp.off_e0);
    e = gbd_launch_onaxis(d_probs, n_runs, sp.rec_stride,
                          precision == GBD_PRECISION_MIXED && sp.algo != GBD_ALGO_RECURRENCE, d_e0, st);
    if (e == cudaSuccess)
        e = gbd_launch_metrics(fields, precision, *det, lambda_fnum, d_e0, d_metrics,
                               reinterpret_cast<double *>(base + sp.off_mpart), n_runs, 10, d_counts, st);
    if (e != cudaSuccess) return cuda_fail(e, "gbd_airy_sweep: on-axis / metrics kernels");
    launches += 3;
    g_launches += launches;
    return done(st, "gbd_airy_sweep (GBD_DEBUG_SYNC)");
}

}  // extern "C"
