// gbd_common.cuh -- shared declarations of the CUDA implementation of libgbd (product code).
// Nothing here is shared with oracle/ (the CPU checker), by design.
#pragma once

#include <cuda_runtime.h>
#include <stdint.h>

#include "../../include/gbd.h"

#define GBD_NREC 13        // physical record, doubles per beamlet (gbd.h)
#define GBD_NEVAL 12       // evaluation record, doubles per beamlet (96 bytes)
#define GBD_NMODE 12       // mode factor of a beamlet: complex a0, a_u, a_v, a_uu, a_uv, a_vv
#define GBD_NEVAL_HG 24    // evaluation record with the mode factor appended

// Rounding constants the pre-pass adds to the constant terms of the detector-coordinate records (GbdFieldLaunch::rec_abs)
// for accumulate_term_fold (gbd_math.cuh explains them)
#define GBD_FOLD_MAGIC_T (6144.0 + 0.001953125)     /* 1.5 * 2^12 + 2^-9 (half a phase-table step) */
#define GBD_FOLD_MAGIC_G 3072.0                     /* 1.5 * 2^11 */
#define GBD_MAGIC_FX_FOLD 6291456.0                 /* 1.5 * 2^22: mixed precision, low word = turns * 2^32 */
#define GBD_FOLD_T_LIMIT 2040.0                     /* |T4| the pre-pass must guarantee (the sum stays in [4096, 8192)) */

// Evaluation record written by the pre-pass (a3 + coefficient scaling), consumed by the field sum.
//   term_j(u,v) = 2^g * (cos 2 pi T + i sin 2 pi T),  Du = u - cu, Dv = v - cv,
//   T4 = 4T = t0 + tu Du + tv Dv + tuu Du^2 + tuv Du Dv + tvv Dv^2       (phase in QUARTER turns)
//   g      = g0 + guu Du^2 + guv Du Dv + gvv Dv^2                         (envelope in log2 units)
// fp64 layout: [cu cv t0 tu tv tuu tuv tvv g0 guu guv gvv].
// mixed layout: the first 8 doubles as above, then 8 floats [g0 guu guv gvv cu cv 0 0].
struct GbdEvalGeom {
    int n_u, n_v;
    double du, dv;          // pixel pitch
    double u0, v0;          // coordinate of pixel index 0: -(n-1)/2 * pitch
};

// One member of a grouped launch (gbd_airy_sweep): several independent field sums on the SAME detector
// evaluated by one persistent kernel; the stream-K partition runs over the concatenated work list.
struct GbdProblem {
    const double *rec;      // evaluation records of this problem
    void *out;              // its [n_v][n_u] field
    long n_b;               // its beamlet count (>= 1)
    long long work_begin;   // first beamlet-tile unit of this problem in the concatenated list
    const double *rec_abs;  // its detector-coordinate records (see GbdFieldLaunch::rec_abs) or NULL
};

struct GbdFieldLaunch {
    const double *rec;      // evaluation records [n_b][12]   (single problem: n_probs == 0)
    long n_b;
    const GbdProblem *probs;   // device table [n_probs] or NULL
    int n_probs;
    long tiles_per_problem;    // = n_tiles when n_probs == 0
    GbdEvalGeom geom;
    int strips_per_row;     // ceil(n_u / (32*P))
    long n_strips;          // n_v * strips_per_row
    long n_tiles;           // ceil(n_strips / warps per CTA), summed over the problems of a grouped launch
    long long work;         // sum over problems of tiles_per_problem * n_b  (beamlet-tile units)
    int slots;              // = gridDim.x of the field-sum kernel
    void *out;              // [n_v][n_u] complex128 or complex64
    void *partial;          // [slots][2][tile_px] complex (same element type as out)
    double log2_tau;        // cull threshold in log2 units (only read by the CULL variants)
    const int *gate;        // device word or NULL: the launch does nothing unless *gate == gate_want (algo 2:
    int gate_want;          // the pre-pass decides on the device which of two enqueued kernels runs)
    const int *deep;        // table kernels: device word or NULL.  0 = the pre-pass found every envelope exponent of
                            // the launch inside [-1000, 1000] on the whole detector, so the exponent clamp is not
                            // needed (and, when rec_abs is given, every beamlet well conditioned in detector
                            // coordinates); NULL / non-zero = take the clamped, beamlet-centred path (always correct)
    const double *rec_abs;  // table kernels, optional: records [n_b][12] of the SAME two quadratics expanded about the
                            // detector centre instead of the beamlet centre,
                            //   [T0 Tu Tv Tuu Tuv Tvv G0 Gu Gv Guu Guv Gvv],  T4 = T0 + Tu u + Tv v + Tuu u^2 + ...,
                            // which saves the Du = u - cu subtraction of every term; only read when *deep == 0
};

// One run of a batched sweep (gbd_airy_sweep): what the lattice, parameter and pre-pass kernels need for it.
struct GbdRunJob {
    int n_across;
    long n;                 // beamlet count (host-computed, = capacity of xy)
    double pitch, r2max;
    double *xy;             // SoA [2][n]
    long *count;            // device count written by the lattice kernel
    double q1_im, lambda, l0_red;
    double *params;         // [n][13]
    double *ev, *ev2;       // evaluation records; ev2: separable layout (algo 2) or NULL
};

// host-side launchers (defined in the .cu files)
cudaError_t gbd_launch_lattice(int n_across, double pitch, double r2max, double *d_xy, long capacity,
                               long *mapped_count, cudaStream_t st);
cudaError_t gbd_launch_propagate(long n, const double *d_xy, long xy_stride, double w0, double lambda,
                                 int abcd_mode, const double *d_abcd, double l0_red,
                                 const double *d_base, const double *d_weight, double *d_params,
                                 cudaStream_t st);
cudaError_t gbd_launch_trace(long n, const double *d_xy, long xy_stride, const double *d_p_in,
                             const double *d_opl0, const gbd_trace_system &S, double lambda, double *d_abcd,
                             double *d_base, cudaStream_t st);
// algo 2 writes 16-double records (evaluation record, S_u, S_v) and sets *d_gate when a beamlet has a cross term
cudaError_t gbd_launch_prepass(long n, const double *d_params, const gbd_detector &det, double lambda,
                               int precision, int algo, double *d_eval, int *d_gate, cudaStream_t st,
                               int *d_deep = nullptr, double *d_eval_abs = nullptr);
cudaError_t gbd_launch_sweep_setup(const GbdRunJob *d_jobs, int n_runs, long max_n, const double *d_abcd,
                                   const gbd_detector &det, int precision, int algo, bool also_separable,
                                   int *d_gate, int *n_launches, cudaStream_t st, int *d_deep = nullptr);
void gbd_sep_geometry(int n_u, int n_v, int precision, int *tiles_u, long *n_tiles);
cudaError_t gbd_launch_field_sep(const GbdFieldLaunch &L, int precision, int *n_launches, cudaStream_t st,
                                 cudaEvent_t ev0, cudaEvent_t ev1);
int gbd_sep_slots(int precision, int sms);
cudaError_t gbd_launch_field(const GbdFieldLaunch &L, int P, int precision, int algo, bool cull,
                             int *n_launches, cudaStream_t st, cudaEvent_t ev0, cudaEvent_t ev1);
cudaError_t gbd_launch_probe(double *d_sink, long iters, double *dfma_per_launch, cudaStream_t st);
// first-order Hermite-Gaussian beamlets (R-23): per-beamlet mode factors, pre-pass and field sum with them
cudaError_t gbd_launch_hg_modes(long n, double w0, double lambda, int abcd_mode, const double *d_abcd,
                                const double *d_mode_weight, double *d_modes, cudaStream_t st);
cudaError_t gbd_launch_prepass_modes(long n, const double *d_params, const double *d_modes, const gbd_detector &det,
                                     double lambda, double *d_eval, cudaStream_t st, int *d_deep = nullptr,
                                     double *d_eval_abs = nullptr);
cudaError_t gbd_launch_field_modes(const GbdFieldLaunch &L, int P, int *n_launches, cudaStream_t st,
                                   cudaEvent_t ev0, cudaEvent_t ev1);
// point-evaluation baseline (gbd_pointeval.cu)
int gbd_pointeval_splits(long n_b, long n_px, int sms);
size_t gbd_pointeval_record_bytes(long n_b);
cudaError_t gbd_launch_pointeval(long n, const double *d_xy, long xy_stride, double w0, double lambda, int abcd_mode,
                                 const double *d_abcd, double l0_red, const double *d_base, const double *d_weight,
                                 const gbd_detector &det, int n_split, double *d_rec, void *d_partial, void *d_field,
                                 int *n_launches, cudaStream_t st, cudaEvent_t ev0, cudaEvent_t ev1);

// error string / launch counter / GBD_DEBUG_SYNC handling of gbd_api.cu, for entry points defined in other files
gbd_status gbd_api_fail(gbd_status code, const char *msg);
gbd_status gbd_api_cuda_fail(cudaError_t e, const char *what);
gbd_status gbd_api_done(cudaStream_t st, int launches, const char *what);
bool gbd_api_detector_ok(const gbd_detector *det);

int gbd_metrics_blocks(long n_px);
// n_runs fields [n_runs][n_v][n_u], e0 [n_runs][2], partials [n_runs][blocks][9], out [n_runs][out_stride];
// d_counts (nullable): per-run beamlet counts copied to out[run][9]
cudaError_t gbd_launch_metrics(const void *d_field, int precision, const gbd_detector &det, double lambda_fnum,
                               const double *d_e0, double *d_out, double *d_part, int n_runs, int out_stride,
                               const long *d_counts, cudaStream_t st);
// on-axis field (detector origin) of n_runs problems: e0[run] = sum_j term_j(0, 0); rec_stride doubles per record
cudaError_t gbd_launch_onaxis(const GbdProblem *d_probs, int n_runs, int rec_stride, int mixed, double *d_e0,
                              cudaStream_t st);

// geometry helpers shared by host and device
__host__ __device__ inline long long gbd_share_begin(long long work, int slots, int s)
{
    return (work * (long long)s) / (long long)slots;
}

void gbd_field_config(int n_u, int precision, int algo, int *P_out, int *threads_out, int *ctas_per_sm_out);
int gbd_field_slots(int precision);
// true when a direct fp64 launch of this plan uses the table kernels (and therefore wants the `deep` word)
bool gbd_field_uses_tables(const GbdFieldLaunch &L, int P, int precision, int algo);
size_t gbd_field_tile_px(int P, int precision);
