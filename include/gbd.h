/*
 * gbd.h -- C ABI of libgbd.so: the plane-evaluation Gaussian Beamlet Decomposition hot path on B200.
 *
 * "P:n" cites /root/reference/PAPER.md line n (arXiv 2404.12454); "R-x" a reading in DESIGN.md.
 *
 * The three calls follow the paper's statement of the problem:
 *   gbd_beamlets_create   decompose the pupil into evenly spaced Gaussian beamlets   P:243-247, Eq. 24
 *   gbd_trace_mirrors     (optional, before the path) 5-ray differential trace -> per-beamlet ABCD
 *   gbd_propagate_q       per-beamlet ABCD -> Q2^-1, amplitude, centre, tilt, path    P:171-177 Eq. 21-22,
 *                                                                                     P:318-320 Eq. 28-29
 *   gbd_eval_field        coherent sum of all beamlets on every detector pixel        P:33 Eq. 3,
 *                         E(r) = sum_j A_j exp(-ik[opl_j + p_j.D + 1/2 D^T Q_j^-1 D]) P:148-157 Eq. 19-20
 *
 * General rules
 *   - Every pointer named d_* is a DEVICE pointer owned by the caller (e.g. a torch tensor's
 *     data_ptr()); it must be 16-byte aligned and outlive the stream work.  Pointers named h_* are
 *     HOST pointers.  The library allocates no device memory; scratch is passed in as a workspace.
 *   - `cuda_stream` is a cudaStream_t (NULL = legacy default stream).  Calls enqueue work and return;
 *     they do not synchronise unless stated (only the *_host call does).
 *   - Units: any consistent length unit (the workloads use mm).  Complex numbers are (re, im) pairs.
 *   - Errors: every call returns a gbd_status; gbd_last_error() gives a thread-local message.
 *     Arguments are validated on the host before any launch.  Asynchronous CUDA faults surface at the
 *     caller's next synchronisation.  There is no CPU fallback: without a CUDA device calls return
 *     GBD_ECUDA.
 *   - fp64 throughout unless precision = 1 is requested in gbd_eval_field.
 *   - Input ranges the kernels assume (not all checkable on the host: the records live on the device).  With
 *     g = log2 of a term's modulus and T its phase in turns anywhere on the detector:
 *       fp64:   |T| < 2^40 turns; any g <= 100 (terms below 2^-1000 are flushed to ~2^-1000 or less); beamlet
 *               amplitudes |A_j| <= 1e30 and a non-growing envelope (Im Q^-1 negative semi-definite), so that g
 *               never exceeds log2 |A_j|.
 *       mixed:  |T| < 2^19 turns (the phase is reduced to a 32-bit fixed-point turn by one fp64 add, exact below
 *               that); g within fp32 range (terms below 2^-126 are flushed to zero).
 *     A beamlet with a non-finite amplitude or one above 1e30 (NaN / Inf weight, singular A + B Q1^-1) makes every pixel NaN; a
 *     beamlet with weight exactly 0 contributes nothing.  Detector pitches and frames must be finite.
 *   - GBD_DEBUG_SYNC=1 in the environment: every call synchronises its stream before returning and reports an
 *     asynchronous fault as its own error; gbd_beamlets_create also reads the lattice kernel's own count back and
 *     compares it with the count the handle carries.
 */
#ifndef GBD_H
#define GBD_H

#include <stddef.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef enum {
    GBD_OK = 0,
    GBD_EINVAL = 1,     /* bad argument (null, misaligned, out of range) */
    GBD_ECAPACITY = 2,  /* caller's buffer / workspace too small */
    GBD_ECUDA = 3,      /* CUDA runtime error (message holds cudaGetErrorString) */
    GBD_ESTATE = 4      /* call order violated (e.g. eval before propagate) */
} gbd_status;

/* Thread-local, never NULL; valid until the next libgbd call on this thread. */
const char *gbd_last_error(void);

/* Number of doubles per beamlet in the parameter record written by gbd_propagate_q (13):
 *   0 c_x 1 c_y | 2 p_x 3 p_y | 4 opl (reduced modulo lambda, R-9) |
 *   5,6 Q_xx | 7,8 Q_xy+Q_yx | 9,10 Q_yy (re,im; Q = Q2^-1, 1/length) | 11,12 amplitude (re,im).
 * Layout: array of structs [n][13], so any run of beamlets is one contiguous byte range. */
int gbd_record_doubles(void);

/* ------------------------------------------------------------------------------------------ a1 */

typedef struct gbd_beamlets gbd_beamlets;   /* opaque; host-side metadata only (n, waist, lambda) */

/* Square lattice of n_across beamlets across `pupil_diameter` (pitch = D/n_across, cell-centred:
 * x_i = (i-(N-1)/2)*pitch), clipped to the circle x^2+y^2 <= (D/2)^2 (R-10); order iy slow, ix fast.
 * waist <= 0 -> waist = overlap_factor*pitch/2 (Eq. 24).
 *   d_xy        out, device, SoA [2][capacity]: x[0..n) then (at offset `capacity`) y[0..n)
 *   capacity    >= number of lattice points kept, else GBD_ECAPACITY (n_across^2 always suffices)
 *   n_out       host, receives n
 * Enqueues one kernel on `cuda_stream` and returns without waiting: n comes from gbd_lattice_count(), which
 * evaluates the kernel's keep/drop predicate in the same individually rounded arithmetic on the host.
 * The caller may afterwards overwrite d_xy in place (jitter, any other layout): the handle keeps
 * only n, the waist and the wavelength. */
gbd_status gbd_beamlets_create(gbd_beamlets **out, int n_across, double pupil_diameter,
                               double overlap_factor, double waist, double wavelength,
                               double *d_xy, long capacity, long *n_out, void *cuda_stream);

/* Same handle for caller-supplied positions (no lattice): n beamlets, explicit waist. */
gbd_status gbd_beamlets_create_custom(gbd_beamlets **out, long n, double waist, double wavelength);

void gbd_beamlets_destroy(gbd_beamlets *);
long gbd_beamlets_count(const gbd_beamlets *);
double gbd_beamlets_waist(const gbd_beamlets *);
double gbd_beamlets_wavelength(const gbd_beamlets *);

/* ------------------------------------------------------------------------------------------ a0 */

/* Differential ray trace: the step BEFORE the path.  "a set of beamlets whose propagation are described
 * by 5 parabasal rays for each beamlet"; "Compute the differential ABCD matrix ... using
 * differential ray tracing" (P:98 step 4).  Each beamlet's base ray and four rays displaced by dq in x,
 * dq in y, dp in p_x, dp in p_y are traced from the pupil plane through up to GBD_MAX_MIRRORS reflecting
 * conics of revolution about z,
 *     c (x^2 + y^2 + (1+k) z'^2) - 2 z' = 0,  z' = z - z_vertex,  c = 1/RoC signed along +z
 * (the standard conic sag; a prescription like P:324-327 Table 2), onto the nominal evaluation plane; the
 * ray-transfer matrix is the forward finite difference of the five rays (refractive index 1).
 *   pupil plane   z = z_pupil, in-plane coordinates = global (x, y); a ray starts at (x_j, y_j) with
 *                 direction (p_x, p_y, dir_sign*sqrt(1-|p|^2)), dir_sign = +1 or -1
 *   evaluation    plane through `origin` spanned by orthonormal e_x, e_y; the light must arrive travelling
 *                 along e_x x e_y.  This frame is the (X, Y, Z) frame of gbd_detector.
 *   d_xy          device SoA [2][xy_stride] beamlet positions
 *   d_p_in        device SoA [2][n] start directions, or NULL (every ray starts along p_common)
 *   d_opl0        device [n] optical path already accumulated at the pupil (field tilt + OPD), or NULL
 *   d_abcd        out, device [n][16] row-major [[A,B],[C,D]] on (q_x,q_y,p_x,p_y)   } exactly what
 *   d_base        out, device SoA [5][n]: q_x, q_y, p_x, p_y on the plane, OPL       } gbd_propagate_q
 *                                                                                      abcd_mode 0 reads
 * The OPL row holds the optical path (d_opl0 + geometric length) REDUCED MODULO THE WAVELENGTH of the handle
 * (fmod: sign of the path, magnitude below lambda; R-24): the field needs the path only modulo lambda, and
 * a double cannot hold a many-metre path to better than ~1e-8 rad of phase, while it holds the remainder exactly.
 * All five rays are traced in double-double arithmetic (~106 bits) and every output is rounded to double once, at
 * the end, so the outputs are the correctly rounded values of the exact trace and the finite differences lose
 * nothing to cancellation.  Needs |path / lambda| < 2^53.  One kernel, no synchronisation. */
#define GBD_MAX_MIRRORS 8
typedef struct {
    double curvature, conic, z_vertex;
} gbd_conic_mirror;
typedef struct {
    int n_mirrors;
    gbd_conic_mirror mirrors[GBD_MAX_MIRRORS];
    double z_pupil, dir_sign;
    double p_common[2];
    double origin[3], e_x[3], e_y[3];
    double dq, dp;
} gbd_trace_system;

gbd_status gbd_trace_mirrors(const gbd_beamlets *, const double *d_xy, long xy_stride,
                             const double *d_p_in, const double *d_opl0, const gbd_trace_system *,
                             double *d_abcd, double *d_base, void *cuda_stream);

/* ------------------------------------------------------------------------------------------ a2 */

/* Per-beamlet complex curvature Q2^-1 = (C + D Q1^-1)(A + B Q1^-1)^-1 (Eq. 22) with
 * Q1^-1 = -i lambda/(pi w0^2) I (R-1), amplitude W/(sqrt(mu1) sqrt(mu2)), mu = eig(A + B Q1^-1)
 * (Eq. 21, branch R-5), centre, tilt and optical path of the base ray; one thread per beamlet.
 *   d_xy       device SoA [2][xy_stride]: beamlet positions r_j in the pupil (used by abcd_mode 1)
 *   abcd_mode  1: d_abcd is ONE row-major 4x4 [[A,B],[C,D]] on (q_x,q_y,p_x,p_y) (Eq. 23);
 *                 d_base is SoA [3][n] = theta_x, theta_y, OPD at the pupil, or NULL (zeros);
 *                 c = A r + B theta, p = C r + D theta (Eq. 28-29),
 *                 path = fmod(l0,lambda) + OPD + 1/2 (p.c - theta.r) (Eq. 17, R-8, R-9).
 *              0: d_abcd is [n][16], one matrix per beamlet (differential ray trace);
 *                 d_base is SoA [5][n] = c_x, c_y, p_x, p_y, OPL of the traced base ray (required; the OPL as
 *                 gbd_trace_mirrors writes it, already reduced, or any full path);
 *                 path = fmod(OPL, lambda); l0 is ignored.
 *   d_weight   SoA [2][n] (re, im) pupil weights W_j, or NULL (1 + 0i)
 *   d_params   out, [n][13] doubles (gbd_params_bytes())                                      */
gbd_status gbd_propagate_q(gbd_beamlets *, const double *d_xy, long xy_stride, int abcd_mode,
                           const double *d_abcd, double l0, const double *d_base,
                           const double *d_weight, double *d_params, void *cuda_stream);
size_t gbd_params_bytes(const gbd_beamlets *);

/* ------------------------------------------------------------------------------------------ a3-a5 */

/* Detector in the frame of the nominal evaluation plane (X, Y in-plane, Z = its normal, z = 0 on it).
 * Pixel (iu, iv) sits at origin + (iu-(n_u-1)/2)*du*e_u + (iv-(n_v-1)/2)*dv*e_v (cell-centred, R-12).
 * e_u, e_v orthonormal.  "Untilted" means e_u = X, e_v = Y and origin z = 0 exactly; anything else
 * takes the tilted-plane re-expansion of DESIGN.md R-T (the paper itself assumes an orthogonal
 * plane). */
typedef struct {
    int n_u, n_v;
    double du, dv;
    double origin[3], e_u[3], e_v[3];
} gbd_detector;

enum { GBD_PRECISION_FP64 = 0, GBD_PRECISION_MIXED = 1 };
enum { GBD_ALGO_DIRECT = 0, GBD_ALGO_RECURRENCE = 1, GBD_ALGO_SEPARABLE = 2 };

/* E[iv][iu] = sum_j (per-term expression above) for every pixel.
 *   d_params   records from gbd_propagate_q
 *   precision  0: fp64 everywhere, output complex128 [n_v][n_u] (re,im interleaved, v slow);
 *              1: phase in fp64, envelope / sincos / accumulation in fp32, output complex64
 *   algo       0: every term evaluated directly (exp2 x sincospi of the fp64 phase);
 *              1: along-row recurrence restarted every 32 (16) pixels: the restart
 *                 values are evaluated as in algo 0, the pixels in between by two complex products each, in
 *                 fp64 (precision 0) or fp32 (precision 1); no cull
 *              2: no cull.  When NO beamlet has a cross term on the detector (Q_uv = 0: rotationally
 *                 symmetric systems on axis) every term factorises into F_j(u) G_j(v) and the sum is evaluated as
 *                 complex rank-1 updates of pixel tiles (4 multiply-adds per term, in fp64 or, precision 1, fp32 with
 *                 the edge values started from the fp64 phase); otherwise the call evaluates
 *                 algo 1.  The decision is taken on the device by the pre-pass (both kernels are enqueued, one
 *                 of them returns at once), so the call still never synchronises
 *   cull_tau   <= 0: off.  > 0: a term whose Gaussian envelope exp((k/2) D^T Im(Q^-1) D) < cull_tau
 *              is dropped, pixel by pixel (R-14)
 *   d_field    out
 *   d_workspace / workspace_bytes   scratch of at least gbd_eval_workspace_bytes()
 * Enqueues: one per-beamlet pre-pass (detector re-expansion + coefficient scaling), the field-sum
 * kernel (persistent, one static work share per CTA), and a small fix-up kernel that adds the
 * partial sums of pixel tiles shared by several CTAs in a fixed order (bitwise reproducible). */
gbd_status gbd_eval_field(const gbd_beamlets *, const double *d_params, const gbd_detector *,
                          int precision, int algo, double cull_tau, void *d_field,
                          void *d_workspace, size_t workspace_bytes, void *cuda_stream);
size_t gbd_eval_workspace_bytes(const gbd_beamlets *, const gbd_detector *, int precision);

/* The whole path a2..a4 with HOST buffers (the end-to-end call): copies h_xy ([2][n]), h_abcd,
 * h_base, h_weight to the device workspace, runs gbd_propagate_q + gbd_eval_field, copies the field
 * to h_field, and synchronises the stream.  Host buffers should be pinned for full PCIe speed.
 * d_workspace must hold gbd_host_workspace_bytes(). */
gbd_status gbd_eval_field_host(gbd_beamlets *, const double *h_xy, int abcd_mode,
                               const double *h_abcd, double l0, const double *h_base,
                               const double *h_weight, const gbd_detector *, int precision, int algo,
                               double cull_tau, void *h_field, void *d_workspace,
                               size_t workspace_bytes, void *cuda_stream);
size_t gbd_host_workspace_bytes(const gbd_beamlets *, const gbd_detector *, int abcd_mode,
                                int precision);

/* ------------------------------------------------------------------------------------------ other beamlet types */

/* Hermite-Gaussian beamlets of orders m + n <= 2 through the same plane-evaluation phasor ("propagation laws
 * for Hermite ... Gaussian beams.  All of these solutions can be employed in beamlet decomposition").  The pupil
 * field of beamlet j is  [sum_{m+n<=2} w_mn H_m(sqrt2 x~/w0) H_n(sqrt2 y~/w0)] exp(-|r~|^2/w0^2) exp(-ik theta.r~),
 * r~ = r1 - r_j, physicists' Hermite polynomials (H0 = 1, H1 = 2 s, H2 = 4 s^2 - 2).  Solving P:82 Eq. 13 with the
 * Hermite generating function (R-23) gives the fundamental term of gbd_eval_field times a complex
 * polynomial of degree <= 2 in D = r - c_j: with M1 = A + B Q1^-1, X = (2 sqrt2/w0)(M1^-1 D)_x, Y likewise, and
 * Gamma = 2 M1^-1 A - I,
 *     factor_j(D) = w00 + w10 X + w01 Y + w20 (X^2 - 2 Gamma_xx) + w11 (X Y - Gamma_xy - Gamma_yx) + w02 (Y^2 - 2 Gamma_yy)
 *                 = a0 + a_x D_x + a_y D_y + a_xx D_x^2 + a_xy D_x D_y + a_yy D_y^2.
 * (Complex weights cover the Laguerre-Gaussian modes of the same orders: LG(p=0, l=+-1) = HG10 +- i HG01,
 * LG(0, +-2) ~ HG20 - HG02 +- 2i HG11, LG(1, 0) = -(HG20 + HG02)/4 -- any fixed linear combination.)
 * gbd_hg_modes computes the factors (one thread per beamlet); gbd_eval_field_modes is gbd_eval_field (fp64, direct
 * algorithm, no cull) with every term multiplied by its factor.  Evaluation planes orthogonal to the axis only:
 * the detector must be untilted (e_u = X, e_v = Y, origin z = 0), the paper's own restriction.
 *   d_abcd, abcd_mode  as for gbd_propagate_q
 *   d_mode_weight      device SoA [12][n]: Re, Im of w00, w10, w01, w20, w11, w02, or NULL (w00 = 1: the
 *                      fundamental beamlet)
 *   d_modes            device [n][12]: Re, Im of a0, a_x, a_y, a_xx, a_xy, a_yy
 *   d_params           records from gbd_propagate_q (the pupil weight W_j multiplies all modes)
 *   d_workspace        >= gbd_eval_modes_workspace_bytes(), 128-byte aligned                              */
gbd_status gbd_hg_modes(const gbd_beamlets *, int abcd_mode, const double *d_abcd, const double *d_mode_weight,
                        double *d_modes, void *cuda_stream);
gbd_status gbd_eval_field_modes(const gbd_beamlets *, const double *d_params, const double *d_modes,
                                const gbd_detector *, void *d_field, void *d_workspace, size_t workspace_bytes,
                                void *cuda_stream);
size_t gbd_eval_modes_workspace_bytes(const gbd_beamlets *, const gbd_detector *);

/* ------------------------------------------------------------------------------------------ baseline */

/* The POINT-evaluation algorithm of P:88-100 (section 2.2, steps 1-6) -- the algorithm the paper's plane
 * evaluation replaces -- kept as a comparison baseline so that the paper's plane / point runtime ratio
 * (Fig. 7) can be restated on one GPU.  For every (pixel, beamlet) pair: distance t = (r_eval - c3).k^ from
 * the base ray's intercept to the transversal plane through the pixel (step 2); the 5 parabasal rays carried there
 * and expressed in its frame (step 3, on the differentials: DESIGN.md R-22); ray-transfer matrix rebuilt on that
 * plane, A' = P0 A + t Pd C, B' = P0 B + t Pd D, C' = Pd C, D' = Pd D (step 4); Gaussian of Eq. 21/22 with that
 * matrix at the pixel's local coordinates xi, E = W / sqrt(det(A' + B' Q1^-1)) exp(-ik [opl + t + 1/2 xi^T Q' xi])
 * (step 5); coherent sum over beamlets (step 6).  The 2x2 complex inverse, eigenvalues and square roots are redone
 * for every pair.  Eq. 21 on the transversal plane normalises power per unit area NORMAL TO THE RAY: the result
 * differs from gbd_eval_field by sqrt(k^.Z) per beamlet (and by the third-order parabasal residual).
 *   d_xy, xy_stride, abcd_mode, d_abcd, l0, d_base, d_weight   exactly as for gbd_propagate_q (which need not
 *              have been called)
 *   detector   as for gbd_eval_field (tilted detectors are simply other 3-D pixel positions here)
 *   d_field    out, [n_v][n_u] complex128
 *   d_workspace >= gbd_pointeval_workspace_bytes(), 256-byte aligned
 * fp64 only.  Three kernels (per-beamlet set-up, field, fixed-order reduction of the beamlet splits); no
 * synchronisation; bitwise reproducible. */
gbd_status gbd_eval_field_pointwise(const gbd_beamlets *, const double *d_xy, long xy_stride, int abcd_mode,
                                    const double *d_abcd, double l0, const double *d_base,
                                    const double *d_weight, const gbd_detector *, void *d_field,
                                    void *d_workspace, size_t workspace_bytes, void *cuda_stream);
size_t gbd_pointeval_workspace_bytes(const gbd_beamlets *, const gbd_detector *);

/* ------------------------------------------------------------------------------------------ metric */

/* Figure of merit of the paper's beamlet-parameter search (Fig. 8-9), computed on the device:
 * I = |E|^2/|E0|^2 against the Airy pattern (2 J1(x)/x)^2, x = pi r/lambda_fnum, r = in-plane distance of
 * the pixel from the detector origin (R-13).
 *   d_field      [n_v][n_u] complex128 (precision 0) or complex64 (1), as written by gbd_eval_field
 *   lambda_fnum  lambda * F# (= the length of one lambda/D on the detector)
 *   d_e0         device, 2 doubles (re, im): the on-axis field used for peak normalisation (a 1x1
 *                gbd_eval_field at the origin)
 *   d_metrics    out, device, 9 doubles: RMS difference over {all pixels, 0-5, 5-10, 10-15 lambda/D},
 *                the four pixel counts, max |I - Airy|
 * Two kernels, deterministic reduction; no synchronisation. */
gbd_status gbd_psf_metrics(const void *d_field, int precision, const gbd_detector *, double lambda_fnum,
                           const double *d_e0, double *d_metrics, void *d_workspace,
                           size_t workspace_bytes, void *cuda_stream);
size_t gbd_psf_metrics_workspace_bytes(const gbd_detector *);

/* gbd_psf_metrics for callers that cannot provide a workspace because they cannot obtain device memory at the point
 * where they need the figure of merit.  Typical cases: a plug-in or pipeline stage that is handed its input and
 * output buffers by a host application which owns all device memory through its own arena (the stage has no
 * allocator handle, and the free HBM outside the arena may be nil, so cudaMalloc would fail); a control loop with a
 * latency budget, where cudaMalloc / cudaFree are ruled out because they take the driver's global lock and may wait
 * for every stream of the device; a long job late in its run, when a fragmented heap makes a fresh allocation a
 * failure mode nobody wants to discover after hours of compute.  Every other call of this library takes its scratch
 * as a caller-owned workspace; this one call takes none.
 *
 * It computes exactly what gbd_psf_metrics computes (same kernels, same block partition, same summation order), for
 * n_fields fields on one detector in one pair of launches.  The block partial sums -- the only scratch the metric
 * needs -- go to an array compiled into the library: GBD_STATIC_METRICS_ROWS rows of 9 doubles = 340,992 bytes of
 * device memory on EVERY GPU on which the process uses libgbd, from the first CUDA call that loads the library's
 * device code there until the process exits, called or not.  The call itself makes no cudaMalloc, cudaFree,
 * cudaHostAlloc or any other allocating call, and uses no memory pool.
 *
 *   d_fields    device, [n_fields][n_v][n_u] complex128 (precision 0) / complex64 (1), contiguous
 *   d_e0        device, [n_fields][2] doubles (re, im): the on-axis value each field is normalised by
 *   d_metrics   out, device, [n_fields][9] doubles, the 9 values of gbd_psf_metrics per field
 *
 * Limit: n_fields * ceil(n_u n_v / 256, capped at 592) must not exceed GBD_STATIC_METRICS_ROWS, i.e. 8 fields of any
 * size (592 rows each from 151,552 px upwards), 74 fields of 128 x 128 px, 4,736 fields of up to 256 px.  A larger
 * request is refused with GBD_ECAPACITY before anything is launched, and gbd_last_error() states the row count asked
 * for and the row count available; split the batch or fall back to gbd_psf_metrics.
 *
 * First call on each device: the call looks up the device address of the built-in array for the CURRENT device
 * (cudaGetSymbolAddress; the host-side name of a device array is not a usable pointer) and remembers it; later calls
 * on that device reuse it.  The device that owns `cuda_stream` must be the current device, as for every launch.  Make
 * that first call during start-up, outside any stream capture.
 *
 * Sharing: all calls on one device use the same array, and it is never cleared -- it need not be, since every row a
 * call reads was written earlier by that same call.  For the same reason two calls that may run on the GPU at the same
 * time (two streams, or two host threads with their own streams) corrupt each other's partial sums: keep the calls of
 * one device on one stream, or order them with events.  Calls on different GPUs are independent.  Enqueues two
 * kernels, no synchronisation. */
#define GBD_STATIC_METRICS_ROWS 4736
gbd_status gbd_psf_metrics_static(const void *d_fields, int n_fields, int precision, const gbd_detector *,
                                  double lambda_fnum, const double *d_e0, double *d_metrics, void *cuda_stream);

/* ------------------------------------------------------------------------------------------ sweep */

/* The paper's beamlet-parameter search ("optimal number of beamlets and overlap factor",
 * Fig. 8; annular zones P:259-269 Fig. 9) as ONE call: for every run r = (beamlets across, pupil
 * diameter, overlap factor, wavelength) the whole path a1..a4 on the same optics (one shared ABCD,
 * abcd_mode 1, unit weights) and the same detector, then the Airy figure of merit of gbd_psf_metrics.
 * The field sums of ALL runs are evaluated by one persistent launch whose stream-K partition runs over
 * the concatenated (run, pixel tile, beamlet) work list, so small runs cannot leave SMs idle; the lattices,
 * parameters, pre-passes, on-axis normalisation values and metrics of all runs take one launch each.  The stream is
 * not synchronised (the three small host tables of the call are uploaded through a process-wide pinned staging
 * buffer; the call waits on the host only if the previous call's upload has not left that buffer yet, and the very
 * first call allocates it).  For that reason the call CANNOT be captured into a CUDA graph: on a capturing stream it
 * returns GBD_ESTATE.  (gbd_beamlets_create, gbd_propagate_q, gbd_eval_field and the other calls can be captured.)
 * The beamlet counts the host needs for planning come from gbd_lattice_count (same individually rounded
 * arithmetic as the lattice kernel, so the two agree bit for bit; the device count is what is reported).
 *   h_runs      host array [n_runs]
 *   d_abcd      device, one row-major 4x4;  l0 its axial path
 *   d_metrics   out, device, [n_runs][10] doubles: the 9 values of gbd_psf_metrics, then the beamlet count
 *   d_fields    out, device, [n_runs][n_v][n_u] complex128 (precision 0) / complex64 (1), or NULL to keep
 *               the fields inside the workspace
 *   d_workspace >= gbd_airy_sweep_workspace_bytes(), 256-byte aligned                                */
typedef struct {
    int n_across;
    double pupil_diameter, overlap_factor, wavelength;
} gbd_sweep_run;

gbd_status gbd_airy_sweep(const gbd_sweep_run *h_runs, int n_runs, const double *d_abcd, double l0,
                          const gbd_detector *, double lambda_fnum, int precision, int algo,
                          double *d_metrics, void *d_fields, void *d_workspace, size_t workspace_bytes,
                          void *cuda_stream);
size_t gbd_airy_sweep_workspace_bytes(const gbd_sweep_run *h_runs, int n_runs, const gbd_detector *,
                                      int precision, int with_fields);

/* Number of lattice points gbd_beamlets_create keeps for (n_across, pupil_diameter); host only, O(N^2). */
long gbd_lattice_count(int n_across, double pupil_diameter);

/* ------------------------------------------------------------------------------------------ misc */

/* FP64-pipe peak probe used by bench.py for the roofline denominator: every thread runs `iters`
 * rounds of 8 independent DFMA chains; grid = 148*8 CTAs x 256 threads.  Returns through
 * *dfma_per_launch the number of thread-level DFMAs one launch executes; the caller times the
 * launch with CUDA events.  d_sink: >= 8 bytes, device. */
gbd_status gbd_probe_dfma(double *d_sink, long iters, double *dfma_per_launch, void *cuda_stream);


/* Total number of kernels libgbd has launched in this process so far (bench.py's gpu_launches is a
 * difference of two readings). */
long gbd_launch_count(void);

/* Profiling hook for bench.py's roofline line: when both are non-NULL (cudaEvent_t), every following
 * gbd_eval_field on this thread records ev_start immediately before and ev_stop immediately after
 * the field-sum kernel launch on the call's stream.  Pass NULLs to switch it off. */
void gbd_set_profile_events(void *ev_start, void *ev_stop);

#ifdef __cplusplus
}
#endif
#endif /* GBD_H */
