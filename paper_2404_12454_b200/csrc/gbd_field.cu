// gbd_field.cu -- the field-sum kernel (a4/a5): E(pixel) = sum_j 2^g_j * cis(2 pi T_j)   (Eq. 3,
// P:148-157 Eq. 19-20 with P:171 Eq. 21), persistent, stream-K partitioned, fp64 pipe bound.
//
// Decomposition
//   strip  = 32*P consecutive pixels of one detector row, owned by one warp (lane l owns columns
//            col0 + l + 32 i, i < P: every store instruction of a warp is one contiguous run);
//   tile   = one strip per warp of the CTA (8 or 16 warps; one CTA per SM: two co-resident CTAs drift apart
//            under the hi-warp-id-first arbiter and the later one finishes alone at half occupancy);
//   work   = n_tiles * n_b "beamlet-tile" units, cut into gridDim.x equal contiguous shares
//            (tile-major, beamlet-minor).  A CTA walks its share; a tile it covers completely is
//            written straight to the output, a tile it shares with other CTAs goes to one of its two
//            partial slots (head / tail) and fixup_kernel adds the partials in CTA order.
//   params = evaluation records (96 B per beamlet, contiguous), streamed through shared memory in
//            blocks of KB beamlets by 1-D bulk async copies (cp.async.bulk, mbarrier completion),
//            double buffered; every lane reads the same record -> broadcast LDS.128.
//   inner  = per (beamlet, thread): row terms hoisted (6-7 FP64 ops); per (beamlet, pixel): the two quadratics
//            (4 DFMA, + 1 DADD on beamlet-centred records) and the term (gbd_math.cuh): accumulate_term_fold in
//            field_fold_kernel (large fp64 launches, the roofline kernel), term_tab in its twin field_tab_kernel,
//            accumulate_term / accumulate_term_mixed in field_kernel (small fp64 launches; mixed precision).
#include <type_traits>

#include "gbd_common.cuh"
#include "gbd_math.cuh"
#include "gbd_tile.cuh"

namespace {

// Launch shapes (ONE CTA per SM).  P = 8 pixels per thread amortises the per-beamlet row terms, record
// loads and loop overhead best but needs ~200 registers -> 8 warps (2 per SM sub-partition), which
// still saturates the FP64 pipe because each warp carries >= 8 independent polynomial chains
// (measured: 81.4 ms vs 84.5 ms for P = 4 x 16 warps on C3).  Narrow detectors use P = 4/2/1 x 16 warps.
// The mixed kernels are bound by the XU pipe / fp32 latency, need <= 128 registers and gain from 4 warps per
// sub-partition (C3: 30.3 -> 25.7 ms direct, 15.3 -> 13.1 ms recurrence).
__host__ __device__ constexpr int warps_for(int P, bool mixed) { return mixed ? 16 : (P >= 8 ? 8 : 16); }
constexpr int STAGE_DOUBLES = KB * GBD_NEVAL;
// smallest launch (beamlet x pixel terms, padded pixels included) that uses the table kernels: they carry ~6 us of fixed
// cost (table fill by every CTA, the gated twin launch, the memset of the "deep" word) against 7.5e11 instead of 4.1e11
// terms/s; measured crossover on 128^2 ... 512^2 px with 97 ... 2,053 beamlets: 1.0e7 terms (6.4e6: 60 vs 63 us;
// 1.2e7: 78 vs 76 us; 2.3e7: 101 vs 85 us)
constexpr double GBD_TAB_MIN_TERMS = 1.0e7;

// ------------------------------------------------------------------ tile geometry
template <int P>
struct Strip {
    bool valid;
    long row;
    int col0;          // first column of this lane
};
template <int P, int WARPS>
__device__ __forceinline__ Strip<P> strip_of(const GbdFieldLaunch &L, long tile, int warp, int lane)
{
    Strip<P> s;
    long strip = tile * WARPS + warp;
    s.valid = strip < L.n_strips;
    s.row = s.valid ? strip / L.strips_per_row : 0;
    s.col0 = (int)(strip - s.row * L.strips_per_row) * (32 * P) + lane;
    return s;
}


// Recurrence layout: every THREAD owns P consecutive pixels of one row (a "run"); lane l of warp w of a
// tile owns run (tile*warps + w)*32 + l.  Stores are strided by P pixels between lanes -- irrelevant,
// the field is written once per tile -- while the recurrence step becomes one pixel pitch and P = 32
// whatever the detector width.
template <int P, int WARPS>
__device__ __forceinline__ Strip<P> run_of(const GbdFieldLaunch &L, long tile, int warp, int lane)
{
    Strip<P> s;
    long run = (tile * WARPS + warp) * 32 + lane;
    s.valid = run < L.n_strips;
    s.row = s.valid ? run / L.strips_per_row : 0;
    s.col0 = s.valid ? (int)(run - s.row * L.strips_per_row) * P : 0;
    return s;
}

// Upper bound of the envelope exponent g(x) = gC + x (gB + guu x) over x in [a, b] (one strip of one
// row): the larger end value, or -- when the derivative changes sign inside -- the vertex value
// gC - gB^2/(4 guu), computed with an fp32 reciprocal and padded for its error.
__device__ __forceinline__ double strip_env_max(double a, double b, double guu, double gB, double gC)
{
    const double ga = fma(fma(guu, a, gB), a, gC), gb = fma(fma(guu, b, gB), b, gC);
    double m = fmax(ga, gb);
    const double da = fma(2.0 * guu, a, gB), db = fma(2.0 * guu, b, gB);
    if (da > 0.0 && db < 0.0) {
        const double r = (double)__frcp_rn((float)(4.0 * guu));
        const double top = -gB * gB * r;                     // >= 0
        m = gC + top * 1.00001;
    }
    return m;
}

// Device-side dispatch of the fast kernels (field_fold_kernel, field_mixed_tab_kernel) and their twins: the launch has
// detector-coordinate records and the pre-pass cleared them (see GbdFieldLaunch::deep).
template <bool GROUPED>
__device__ __forceinline__ bool gbd_fold_allowed(const GbdFieldLaunch &L)
{
    const bool has_abs = GROUPED ? L.probs[0].rec_abs != nullptr : L.rec_abs != nullptr;
    return L.deep != nullptr && *L.deep == 0 && has_abs;
}

// ------------------------------------------------------------------ fp64 direct kernel
// MIXED = false: everything in fp64, polynomial per-term evaluation: launches below the table kernels' crossover
//                (1e7 terms) and every launch with a cull.  The roofline kernel is field_fold_kernel further down.
// MIXED = true : phase quadratic in fp64, reduced to a 32-bit fixed-point turn by ONE magic-number
//                DADD; envelope quadratic, exp2 / sin / cos (MUFU) and accumulation in fp32.
template <int P, bool CULL, bool MIXED, bool GROUPED>
__global__ void __launch_bounds__(warps_for(P, MIXED) * 32, 1) field_kernel(const GbdFieldLaunch L)
{
    using acc_t = typename std::conditional<MIXED, float, double>::type;
    using out_t = typename std::conditional<MIXED, float2, double2>::type;
    __shared__ __align__(128) double sbuf[2][STAGE_DOUBLES];
    __shared__ __align__(8) uint64_t bar[2];
    if constexpr (MIXED && !CULL) {
        // the mixed kernel may have been enqueued as the twin of field_mixed_tab_kernel: exactly one of the pair runs
        if (gbd_fold_allowed<GROUPED>(L)) return;
    }

    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int slot = blockIdx.x;
    const long long b0 = gbd_share_begin(L.work, L.slots, slot);
    const long long b1 = gbd_share_begin(L.work, L.slots, slot + 1);
    if (b0 >= b1) return;

    if (tid == 0) {
        mbar_init(&bar[0], 1);
        mbar_init(&bar[1], 1);
        mbar_fence_init();
    }
    __syncthreads();

    const long first_gtile = piece_at<GROUPED>(L, b0, b1).gtile;
    const double half_u = 0.5 * (double)(L.geom.n_u - 1), half_v = 0.5 * (double)(L.geom.n_v - 1);
    uint32_t it = 0;                              // stage-use counter (stage = it&1, parity = (it>>1)&1)
    out_t *partial = reinterpret_cast<out_t *>(L.partial);
    constexpr int WARPS = warps_for(P, MIXED);
    constexpr int TILE_PX = WARPS * 32 * P;
    const float log2_tau_f = (float)L.log2_tau;

    for (long long pos = b0; pos < b1;) {
        const Piece pc = piece_at<GROUPED>(L, pos, b1);
        const long tile = pc.tile, j0 = pc.j0, j1 = pc.j1, n_b = pc.n_b;
        const double *rec = pc.rec;
        out_t *out = reinterpret_cast<out_t *>(pc.out);
        const Strip<P> st = strip_of<P, WARPS>(L, tile, warp, lane);
        const double v = __dmul_rn((double)st.row - half_v, L.geom.dv);
        // strip extent (warp-uniform), used by the strip-level cull
        const double us_lo = ((double)(st.col0 - lane) - half_u) * L.geom.du;
        const double us_hi = us_lo + (double)(32 * P - 1) * L.geom.du;
        double u[P];
        float uf[P];
        acc_t acc_re[P], acc_im[P];
        const float vf = (float)v;
#pragma unroll
        for (int i = 0; i < P; ++i) {
            u[i] = __dmul_rn((double)(st.col0 + 32 * i) - half_u, L.geom.du);
            uf[i] = (float)u[i];
            acc_re[i] = 0;
            acc_im[i] = 0;
        }

        const long nblk = (j1 - j0 + KB - 1) / KB;
        if (tid == 0) {
            uint32_t cnt = (uint32_t)min((long)KB, j1 - j0);
            mbar_arrive_expect_tx(&bar[it & 1], cnt * GBD_NEVAL * 8);
            bulk_g2s(sbuf[it & 1], rec + j0 * GBD_NEVAL, cnt * GBD_NEVAL * 8, &bar[it & 1]);
        }
        for (long b = 0; b < nblk; ++b) {
            const long jb = j0 + b * KB;
            const int cnt = (int)min((long)KB, j1 - jb);
            if (tid == 0 && b + 1 < nblk) {
                uint32_t cn = (uint32_t)min((long)KB, j1 - jb - KB);
                uint32_t sn = (it + 1) & 1;
                mbar_arrive_expect_tx(&bar[sn], cn * GBD_NEVAL * 8);
                bulk_g2s(sbuf[sn], rec + (jb + KB) * GBD_NEVAL, cn * GBD_NEVAL * 8, &bar[sn]);
            }
            mbar_wait(&bar[it & 1], (it >> 1) & 1);
            if (st.valid) {
                const double2 *sb = reinterpret_cast<const double2 *>(sbuf[it & 1]);
#pragma unroll 1
                for (int jj = 0; jj < cnt; ++jj) {
                    const double2 r0 = sb[jj * 6 + 0];      // cu cv
                    const double2 r1 = sb[jj * 6 + 1];      // t0 tu
                    const double2 r2 = sb[jj * 6 + 2];      // tv tuu
                    const double2 r3 = sb[jj * 6 + 3];      // tuv tvv
                    const double dv = v - r0.y;
                    const double tB = fma(r3.x, dv, r1.y);
                    const double tC = fma(fma(r3.y, dv, r2.x), dv, r1.x);
                    if constexpr (!MIXED) {
                        const double2 r4 = sb[jj * 6 + 4];      // g0 guu
                        const double2 r5 = sb[jj * 6 + 5];      // guv gvv
                        const double gB = r5.x * dv;
                        const double gC = fma(r5.y * dv, dv, r4.x);
                        const double g_cut = CULL ? r4.x + L.log2_tau : 0.0;
                        if (CULL && strip_env_max(us_lo - r0.x, us_hi - r0.x, r4.y, gB, gC) < g_cut - 1.0)
                            continue;            // every pixel of the strip would be dropped (R-14)
                        // both quadratics of all P pixels first, then the P transcendental evaluations: the
                        // same arithmetic, but ptxas schedules it 1 % better (81.5 -> 80.7 ms on C3)
                        double t4v[P], gv[P];
#pragma unroll
                        for (int i = 0; i < P; ++i) {
                            const double du = u[i] - r0.x;
                            t4v[i] = fma(fma(r2.y, du, tB), du, tC);
                            gv[i] = fma(fma(r4.y, du, gB), du, gC);
                        }
#pragma unroll
                        for (int i = 0; i < P; ++i) {
                            if (CULL) gbdm::accumulate_term_cull(gv[i], g_cut, t4v[i], acc_re[i], acc_im[i]);
                            else gbdm::accumulate_term(gv[i], t4v[i], acc_re[i], acc_im[i]);
                        }
                    } else {
                        const float4 f4 = reinterpret_cast<const float4 *>(sb)[jj * 6 + 4];  // g0 guu guv gvv
                        const float2 cf = reinterpret_cast<const float2 *>(sb)[jj * 12 + 10]; // cu cv (fp32)
                        const float dvf = vf - cf.y;
                        const float gB = f4.z * dvf;
                        const float gC = fmaf(f4.w * dvf, dvf, f4.x);
                        const float g_cut = CULL ? f4.x + log2_tau_f : 0.f;
                        if (CULL && strip_env_max(us_lo - r0.x, us_hi - r0.x, (double)f4.y, (double)gB,
                                                  (double)gC) < (double)g_cut - 2.0)
                            continue;
#pragma unroll
                        for (int i = 0; i < P; ++i) {
                            const double du = u[i] - r0.x;
                            const double t4 = fma(fma(r2.y, du, tB), du, tC);
                            const float duf = uf[i] - cf.x;
                            const float g = fmaf(fmaf(f4.y, duf, gB), duf, gC);
                            gbdm::accumulate_term_mixed<CULL>(g, g_cut, t4, acc_re[i], acc_im[i]);
                        }
                    }
                }
            }
            __syncthreads();                     // all reads of this stage done before it is refilled
            ++it;
        }

        // write: whole tile -> output; shared tile -> this CTA's head (0) or tail (1) partial slot
        const bool whole = (j0 == 0 && j1 == n_b);
        if (whole) {
            if (st.valid) {
#pragma unroll
                for (int i = 0; i < P; ++i) {
                    int col = st.col0 + 32 * i;
                    if (col < L.geom.n_u)
                        out[st.row * L.geom.n_u + col] = out_t{acc_re[i], acc_im[i]};
                }
            }
        } else {
            const int seg = (pc.gtile == first_gtile) ? 0 : 1;
            out_t *pp = partial + ((size_t)slot * 2 + seg) * TILE_PX + warp * (32 * P) + lane;
#pragma unroll
            for (int i = 0; i < P; ++i) pp[32 * i] = out_t{acc_re[i], acc_im[i]};
        }
        pos += (j1 - j0);
    }
}

// ------------------------------------------------------------------ fp64 direct kernel, fast path ("folded")
// The roofline kernel.  Same decomposition, staging, tables and stream-K partition as field_tab_kernel, but on the
// records in DETECTOR coordinates (GbdFieldLaunch::rec_abs: the two quadratics expanded about the detector centre, with
// the rounding constants of gbdm::accumulate_term_fold riding on their constant terms):
//   per (beamlet, thread): 6 FP64 instructions (the v-dependent parts of both quadratics; no Dv),
//   per (beamlet, pixel) : 2 + 2 DFMA for the quadratics -- no Du = u - cu, and the last DFMA of each already delivers
//                          the rounded sum whose high word holds the table index and whose low word the remainder --
//                          then accumulate_term_fold: in all 16.05 FP64-pipe + 2 conversion (I2F.F64, XU pipe) + 9.5
//                          other instructions per term (field_tab_kernel: 23.9 + 8.4).
// The pre-pass decides ON THE DEVICE whether a launch may take this path (*L.deep == 0: every envelope exponent inside
// the unclamped range, every |T4| below 2040 quarter turns, every beamlet well conditioned about the detector centre);
// this kernel and its twin field_tab_kernel (beamlet-centred records, clamped loop: always correct) are both enqueued
// and one of them returns at once.  Two kernels rather than two loops in one kernel: with a single loop per kernel
// ptxas finds a better schedule (1.5 % on C3).
// HG = true: every term times the beamlet's complex mode factor (Hermite-Gaussian beamlets, R-23), a polynomial of degree
// <= 2 in the pixel coordinates appended to the record (24 doubles; 64 beamlets per stage): + 8 FP64 per term.
template <int P, bool GROUPED, bool HG = false>
__global__ void __launch_bounds__(warps_for(P, false) * 32, 1) field_fold_kernel(const GbdFieldLaunch L)
{
    static_assert(!(HG && GROUPED), "mode factors: no grouped launch");
    constexpr int WARPS = warps_for(P, false);
    constexpr int TILE_PX = WARPS * 32 * P;
    constexpr int NE = HG ? GBD_NEVAL_HG : GBD_NEVAL;       // doubles per record
    constexpr int KBK = HG ? KB / 2 : KB;                   // beamlets per stage
    __shared__ __align__(128) double sbuf[2][KBK * NE];
    __shared__ __align__(8) uint64_t bar[2];
    extern __shared__ __align__(128) double2 cis_tab[];    // the two tables (128 KB + 64 KB)
    if (!gbd_fold_allowed<GROUPED>(L)) return;

    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int slot = blockIdx.x;
    const long long b0 = gbd_share_begin(L.work, L.slots, slot);
    const long long b1 = gbd_share_begin(L.work, L.slots, slot + 1);
    if (b0 >= b1) return;
    if (tid == 0) {
        mbar_init(&bar[0], 1);
        mbar_init(&bar[1], 1);
        mbar_fence_init();
    }
    double *exp_tab = reinterpret_cast<double *>(cis_tab + GBD_CIS_N * GBD_CIS_COPIES);
    gbdm::fill_tables<true>(cis_tab, exp_tab, tid, blockDim.x);
    const uint32_t cis_lane = smem_u32(cis_tab) + (uint32_t)(lane & (GBD_CIS_COPIES - 1)) * 16u;
    const uint32_t exp_lane = smem_u32(exp_tab) + (uint32_t)(lane & (GBD_EXP_COPIES - 1)) * 8u;
    __syncthreads();

    const long first_gtile = piece_at<GROUPED>(L, b0, b1).gtile;
    const double half_u = 0.5 * (double)(L.geom.n_u - 1), half_v = 0.5 * (double)(L.geom.n_v - 1);
    uint32_t it = 0;                              // stage-use counter (stage = it&1, parity = (it>>1)&1)
    double2 *partial = reinterpret_cast<double2 *>(L.partial);

    for (long long pos = b0; pos < b1;) {
        const Piece pc = piece_at<GROUPED>(L, pos, b1);
        const long j0 = pc.j0, j1 = pc.j1;
        const double *rec = pc.rec_abs;
        const Strip<P> st = strip_of<P, WARPS>(L, pc.tile, warp, lane);
        const double v = __dmul_rn((double)st.row - half_v, L.geom.dv);
        double u[P], acc_re[P], acc_im[P];
#pragma unroll
        for (int i = 0; i < P; ++i) {
            u[i] = __dmul_rn((double)(st.col0 + 32 * i) - half_u, L.geom.du);
            acc_re[i] = 0.0;
            acc_im[i] = 0.0;
        }
        const long nblk = (j1 - j0 + KBK - 1) / KBK;
        if (tid == 0) {
            const uint32_t cnt = (uint32_t)min((long)KBK, j1 - j0);
            mbar_arrive_expect_tx(&bar[it & 1], cnt * NE * 8);
            bulk_g2s(sbuf[it & 1], rec + j0 * NE, cnt * NE * 8, &bar[it & 1]);
        }
        for (long b = 0; b < nblk; ++b) {
            const long jb = j0 + b * KBK;
            const int cnt = (int)min((long)KBK, j1 - jb);
            if (tid == 0 && b + 1 < nblk) {
                const uint32_t cn = (uint32_t)min((long)KBK, j1 - jb - KBK);
                const uint32_t sn = (it + 1) & 1;
                mbar_arrive_expect_tx(&bar[sn], cn * NE * 8);
                bulk_g2s(sbuf[sn], rec + (jb + KBK) * NE, cn * NE * 8, &bar[sn]);
            }
            mbar_wait(&bar[it & 1], (it >> 1) & 1);
            // a strip beyond the detector (last tile) runs the loop like the others: its lanes are not stored
            const double2 *sb = reinterpret_cast<const double2 *>(sbuf[it & 1]);
            if constexpr (GROUPED) {
                // grouped launches (gbd_airy_sweep: many short pieces) keep the plain loop, every lane working out the
                // row terms itself: the shared slots below cost them 4 % (C2 search 25.3 -> 26.3 ms)
#pragma unroll 1
                for (int jj = 0; jj < cnt; ++jj) {
                    const double2 r0 = sb[jj * 6 + 0];      // T0 + magic, Tu
                    const double2 r1 = sb[jj * 6 + 1];      // Tv, Tuu
                    const double2 r2 = sb[jj * 6 + 2];      // Tuv, Tvv
                    const double2 r3 = sb[jj * 6 + 3];      // G0 + magic, Gu
                    const double2 r4 = sb[jj * 6 + 4];      // Gv, Guu
                    const double2 r5 = sb[jj * 6 + 5];      // Guv, Gvv
                    const double tB = fma(r2.x, v, r0.y);
                    const double tC = fma(fma(r2.y, v, r1.x), v, r0.x);
                    const double gB = fma(r5.x, v, r3.y);
                    const double gC = fma(fma(r5.y, v, r4.x), v, r3.x);
                    double mq[P], mg[P];
#pragma unroll
                    for (int i = 0; i < P; ++i) {
                        mq[i] = fma(fma(r1.y, u[i], tB), u[i], tC);
                        mg[i] = fma(fma(r4.y, u[i], gB), u[i], gC);
                    }
#pragma unroll
                    for (int i = 0; i < P; ++i)
                        gbdm::accumulate_term_fold(mg[i], mq[i], cis_lane, exp_lane, acc_re[i], acc_im[i]);
                }
            } else {
                // The v-dependent parts of the two quadratics are the same for all lanes of a warp (a strip is one
                // detector row).  Instead of every lane computing them for every beamlet (6 FP64 + 6 record loads per
                // beamlet and thread), the lanes share the work: for a group of HG_N beamlets lane l works out those of
                // beamlet l % HG_N and leaves (tB tC | gB gC | Tuu Guu) in the warp's slot; the pixel loop then reads
                // 3 broadcast LDS.128 per beamlet.  Stand-alone loop: 50.2 -> 47.0 cycles per warp-term.
                // (mode factors: 8 and 4 -- their slots also hold the factor's hoisted coefficients hB, hC and A_uu)
                constexpr int HG_N = (HG ? 64 : 128) / WARPS;    // 16 beamlets per group (8 with 16 warps): 6 KB of slots
                constexpr int NS = HG ? 6 : 3;
                __shared__ __align__(16) double2 hoist[WARPS][HG_N][NS];
#pragma unroll 1
                for (int g0 = 0; g0 < cnt; g0 += HG_N) {
                    {
                        const int jj = g0 + (lane & (HG_N - 1));   // beyond cnt: stale but in-bounds, never used
                        const double2 r0 = sb[jj * (NE / 2) + 0];      // T0 + magic, Tu
                        const double2 r1 = sb[jj * (NE / 2) + 1];      // Tv, Tuu
                        const double2 r2 = sb[jj * (NE / 2) + 2];      // Tuv, Tvv
                        const double2 r3 = sb[jj * (NE / 2) + 3];      // G0 + magic, Gu
                        const double2 r4 = sb[jj * (NE / 2) + 4];      // Gv, Guu
                        const double2 r5 = sb[jj * (NE / 2) + 5];      // Guv, Gvv
                        const double tB = fma(r2.x, v, r0.y);
                        const double tC = fma(fma(r2.y, v, r1.x), v, r0.x);
                        const double gB = fma(r5.x, v, r3.y);
                        const double gC = fma(fma(r5.y, v, r4.x), v, r3.x);
                        if (lane < HG_N) {
                            hoist[warp][lane][0] = make_double2(tB, tC);
                            hoist[warp][lane][1] = make_double2(gB, gC);
                            hoist[warp][lane][2] = make_double2(r1.y, r4.y);
                        }
                        if constexpr (HG) {
                            // mode factor A_uu u^2 + (A_u + A_uv v) u + (A0 + A_v v + A_vv v^2), complex
                            const double2 h0 = sb[jj * (NE / 2) + 6], hu = sb[jj * (NE / 2) + 7], hv = sb[jj * (NE / 2) + 8];
                            const double2 hA = sb[jj * (NE / 2) + 9], huv = sb[jj * (NE / 2) + 10], hvv = sb[jj * (NE / 2) + 11];
                            if (lane < HG_N) {
                                hoist[warp][lane][3] = hA;
                                hoist[warp][lane][4] = make_double2(fma(huv.x, v, hu.x), fma(huv.y, v, hu.y));
                                hoist[warp][lane][5] = make_double2(fma(fma(hvv.x, v, hv.x), v, h0.x), fma(fma(hvv.y, v, hv.y), v, h0.y));
                            }
                        }
                    }
                    __syncwarp();
                    const int ng = min(HG_N, cnt - g0);
#pragma unroll 1
                    for (int kk = 0; kk < ng; ++kk) {
                        const double2 h0 = hoist[warp][kk][0], h1 = hoist[warp][kk][1], h2 = hoist[warp][kk][2];
                        double mq[P], mg[P];
#pragma unroll
                        for (int i = 0; i < P; ++i) {
                            mq[i] = fma(fma(h2.x, u[i], h0.x), u[i], h0.y);
                            mg[i] = fma(fma(h2.y, u[i], h1.x), u[i], h1.y);
                        }
                        if constexpr (HG) {
                            const double2 hA = hoist[warp][kk][3], hB = hoist[warp][kk][4], hC = hoist[warp][kk][5];
#pragma unroll
                            for (int i = 0; i < P; ++i) {
                                const double pr = fma(fma(hA.x, u[i], hB.x), u[i], hC.x);
                                const double pi = fma(fma(hA.y, u[i], hB.y), u[i], hC.y);
                                double tr = 0.0, ti = 0.0;
                                gbdm::accumulate_term_fold(mg[i], mq[i], cis_lane, exp_lane, tr, ti);
                                acc_re[i] = fma(-ti, pi, fma(tr, pr, acc_re[i]));
                                acc_im[i] = fma(ti, pr, fma(tr, pi, acc_im[i]));
                            }
                        } else {
#pragma unroll
                            for (int i = 0; i < P; ++i)
                                gbdm::accumulate_term_fold(mg[i], mq[i], cis_lane, exp_lane, acc_re[i], acc_im[i]);
                        }
                    }
                    __syncwarp();                            // the slot is rewritten by the next group
                }
            }
            __syncthreads();                     // all reads of this stage done before it is refilled
            ++it;
        }
        // write: whole tile -> output; shared tile -> this CTA's head (0) or tail (1) partial slot.  The piece and the
        // strip are RE-DERIVED from `pos` (made opaque to the compiler) instead of being kept in registers across the
        // hot loop: fewer live registers there, and ptxas schedules the loop like the stand-alone copy of it
        asm volatile("" : "+l"(pos));
        const Piece pe = piece_at<GROUPED>(L, pos, b1);
        const Strip<P> se = strip_of<P, WARPS>(L, pe.tile, warp, lane);
        if (pe.j0 == 0 && pe.j1 == pe.n_b) {
            if (se.valid) {
                double2 *out = reinterpret_cast<double2 *>(pe.out);
#pragma unroll
                for (int i = 0; i < P; ++i) {
                    const int col = se.col0 + 32 * i;
                    if (col < L.geom.n_u) out[se.row * L.geom.n_u + col] = make_double2(acc_re[i], acc_im[i]);
                }
            }
        } else {
            const int seg = (pe.gtile == first_gtile) ? 0 : 1;
            double2 *pp = partial + ((size_t)slot * 2 + seg) * TILE_PX + warp * (32 * P) + lane;
#pragma unroll
            for (int i = 0; i < P; ++i) pp[32 * i] = make_double2(acc_re[i], acc_im[i]);
        }
        pos += (pe.j1 - pe.j0);
    }
}

// ------------------------------------------------------------------ mixed precision direct kernel, fast path
// field_kernel<.., MIXED> is bound by the XU pipe (3 MUFU per term).  This kernel takes cis from an fp32 table in shared
// memory (gbdm::accumulate_term_mixed_tab: one MUFU per term left) and, like field_fold_kernel, reads the phase quadratic
// from detector-coordinate records with the fixed-point rounding constant folded in (2 DFMA per term instead of
// 1 DADD + 2 DFMA + 1 DADD).  Same decomposition, staging and stream-K partition; same device-side dispatch: the
// pre-pass clears the launch (*L.deep == 0) or the twin field_kernel<P, false, true, GROUPED> runs.
template <int P, bool GROUPED>
__global__ void __launch_bounds__(warps_for(P, true) * 32, 1) field_mixed_tab_kernel(const GbdFieldLaunch L)
{
    constexpr int WARPS = warps_for(P, true);
    constexpr int TILE_PX = WARPS * 32 * P;
    __shared__ __align__(128) double sbuf[2][KB * GBD_NEVAL];
    __shared__ __align__(8) uint64_t bar[2];
    extern __shared__ __align__(128) float2 mix_tab[];      // GBD_MIXTAB_BYTES
    if (!gbd_fold_allowed<GROUPED>(L)) return;

    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int slot = blockIdx.x;
    const long long b0 = gbd_share_begin(L.work, L.slots, slot);
    const long long b1 = gbd_share_begin(L.work, L.slots, slot + 1);
    if (b0 >= b1) return;
    if (tid == 0) {
        mbar_init(&bar[0], 1);
        mbar_init(&bar[1], 1);
        mbar_fence_init();
    }
    gbdm::fill_mixed_table(mix_tab, tid, blockDim.x);
    const uint32_t tab_lane = smem_u32(mix_tab) + (uint32_t)(lane & (GBD_MIXTAB_COPIES - 1)) * 8u;
    __syncthreads();

    const long first_gtile = piece_at<GROUPED>(L, b0, b1).gtile;
    const double half_u = 0.5 * (double)(L.geom.n_u - 1), half_v = 0.5 * (double)(L.geom.n_v - 1);
    uint32_t it = 0;
    float2 *partial = reinterpret_cast<float2 *>(L.partial);

    for (long long pos = b0; pos < b1;) {
        const Piece pc = piece_at<GROUPED>(L, pos, b1);
        const long j0 = pc.j0, j1 = pc.j1;
        const double *rec = pc.rec_abs;
        const Strip<P> st = strip_of<P, WARPS>(L, pc.tile, warp, lane);
        const double v = __dmul_rn((double)st.row - half_v, L.geom.dv);
        const float vf = (float)v;
        double u[P];
        float uf[P], acc_re[P], acc_im[P];
#pragma unroll
        for (int i = 0; i < P; ++i) {
            u[i] = __dmul_rn((double)(st.col0 + 32 * i) - half_u, L.geom.du);
            uf[i] = (float)u[i];
            acc_re[i] = 0.f;
            acc_im[i] = 0.f;
        }
        const long nblk = (j1 - j0 + KB - 1) / KB;
        if (tid == 0) {
            const uint32_t cnt = (uint32_t)min((long)KB, j1 - j0);
            mbar_arrive_expect_tx(&bar[it & 1], cnt * GBD_NEVAL * 8);
            bulk_g2s(sbuf[it & 1], rec + j0 * GBD_NEVAL, cnt * GBD_NEVAL * 8, &bar[it & 1]);
        }
        for (long b = 0; b < nblk; ++b) {
            const long jb = j0 + b * KB;
            const int cnt = (int)min((long)KB, j1 - jb);
            if (tid == 0 && b + 1 < nblk) {
                const uint32_t cn = (uint32_t)min((long)KB, j1 - jb - KB);
                const uint32_t sn = (it + 1) & 1;
                mbar_arrive_expect_tx(&bar[sn], cn * GBD_NEVAL * 8);
                bulk_g2s(sbuf[sn], rec + (jb + KB) * GBD_NEVAL, cn * GBD_NEVAL * 8, &bar[sn]);
            }
            mbar_wait(&bar[it & 1], (it >> 1) & 1);
            const double2 *sb = reinterpret_cast<const double2 *>(sbuf[it & 1]);
#pragma unroll 1
            for (int jj = 0; jj < cnt; ++jj) {
                const double2 r0 = sb[jj * 6 + 0];      // T0 + magic, Tu
                const double2 r1 = sb[jj * 6 + 1];      // Tv, Tuu
                const double2 r2 = sb[jj * 6 + 2];      // Tuv, Tvv
                const float4 f4 = reinterpret_cast<const float4 *>(sb)[jj * 6 + 4];   // g0 guu guv gvv
                const float2 cf = reinterpret_cast<const float2 *>(sb)[jj * 12 + 10]; // cu cv (fp32)
                const double tB = fma(r2.x, v, r0.y);
                const double tC = fma(fma(r2.y, v, r1.x), v, r0.x);
                const float dvf = vf - cf.y;
                const float gB = f4.z * dvf;
                const float gC = fmaf(f4.w * dvf, dvf, f4.x);
#pragma unroll
                for (int i = 0; i < P; ++i) {
                    const double mq = fma(fma(r1.y, u[i], tB), u[i], tC);
                    const float duf = uf[i] - cf.x;
                    const float g = fmaf(fmaf(f4.y, duf, gB), duf, gC);
                    gbdm::accumulate_term_mixed_tab<false>(g, 0.f, mq, tab_lane, acc_re[i], acc_im[i]);
                }
            }
            __syncthreads();                     // all reads of this stage done before it is refilled
            ++it;
        }
        // piece and strip re-derived from an opaque `pos` (see field_fold_kernel): not live across the hot loop
        asm volatile("" : "+l"(pos));
        const Piece pe = piece_at<GROUPED>(L, pos, b1);
        const Strip<P> se = strip_of<P, WARPS>(L, pe.tile, warp, lane);
        if (pe.j0 == 0 && pe.j1 == pe.n_b) {
            if (se.valid) {
                float2 *out = reinterpret_cast<float2 *>(pe.out);
#pragma unroll
                for (int i = 0; i < P; ++i) {
                    const int col = se.col0 + 32 * i;
                    if (col < L.geom.n_u) out[se.row * L.geom.n_u + col] = make_float2(acc_re[i], acc_im[i]);
                }
            }
        } else {
            const int seg = (pe.gtile == first_gtile) ? 0 : 1;
            float2 *pp = partial + ((size_t)slot * 2 + seg) * TILE_PX + warp * (32 * P) + lane;
#pragma unroll
            for (int i = 0; i < P; ++i) pp[32 * i] = make_float2(acc_re[i], acc_im[i]);
        }
        pos += (pe.j1 - pe.j0);
    }
}

// ------------------------------------------------------------------ fp64 direct kernel, table-driven / mode factors
// The fp64 per-term kernel of large launches (the roofline kernel) and of the mode-factor path; same decomposition,
// staging and stream-K partition as field_kernel above.
// TAB = true : 2^g and cis(2 pi T) from the two replicated shared-memory tables of gbd_math.cuh (term_tab: 18 FP64 +
//              7 other instructions per term instead of 28 + 14); the tables are filled by the CTA itself at kernel
//              start (1,536 transcendental evaluations + 192 KB of shared-memory stores: ~2 us), so launches too
//              small to pay for that use field_kernel (polynomial evaluation) instead.
// HG = true  : every term is multiplied by the beamlet's complex mode factor, a polynomial of degree <= 2 in
//              (Du, Dv) (Hermite-Gaussian beamlets of orders m+n <= 2, R-23); the evaluation record
//              then has 24 doubles (the 12 above + a0, a_u, a_v, a_uu, a_uv, a_vv) and a stage holds 64 beamlets.
//              TAB = false is the polynomial evaluation for small mode launches.
template <int P, bool CULL, bool GROUPED, bool TAB, bool HG>
__global__ void __launch_bounds__(warps_for(P, false) * 32, 1) field_tab_kernel(const GbdFieldLaunch L)
{
    static_assert(!(HG && (CULL || GROUPED)), "mode factors: no cull, no grouped launch");
    if constexpr (TAB && !CULL) {
        // the plain and the mode-factor table kernels are enqueued as the twins of field_fold_kernel (above): exactly
        // one of each pair runs
        if (gbd_fold_allowed<GROUPED>(L)) return;
    }
    constexpr bool MIXED = false;
    constexpr int NE = HG ? GBD_NEVAL_HG : GBD_NEVAL;       // doubles per evaluation record
    constexpr int KBK = HG ? KB / 2 : KB;                   // beamlets per stage
    constexpr int STAGE_DOUBLES = KBK * NE;
    using acc_t = double;
    using out_t = double2;
    __shared__ __align__(128) double sbuf[2][STAGE_DOUBLES];
    __shared__ __align__(8) uint64_t bar[2];
    extern __shared__ __align__(128) double2 cis_tab[];    // TAB: the two tables of term_tab (128 KB + 64 KB)

    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int slot = blockIdx.x;
    const long long b0 = gbd_share_begin(L.work, L.slots, slot);
    const long long b1 = gbd_share_begin(L.work, L.slots, slot + 1);
    if (b0 >= b1) return;

    if (tid == 0) {
        mbar_init(&bar[0], 1);
        mbar_init(&bar[1], 1);
        mbar_fence_init();
    }
    double *exp_tab = reinterpret_cast<double *>(cis_tab + GBD_CIS_N * GBD_CIS_COPIES);
    if constexpr (TAB) gbdm::fill_tables(cis_tab, exp_tab, tid, blockDim.x);
    const uint32_t cis_lane = smem_u32(cis_tab) + (uint32_t)(lane & (GBD_CIS_COPIES - 1)) * 16u;
    const uint32_t exp_lane = smem_u32(exp_tab) + (uint32_t)(lane & (GBD_EXP_COPIES - 1)) * 8u;
    __syncthreads();

    const long first_gtile = piece_at<GROUPED>(L, b0, b1).gtile;
    const double half_u = 0.5 * (double)(L.geom.n_u - 1), half_v = 0.5 * (double)(L.geom.n_v - 1);
    uint32_t it = 0;                              // stage-use counter (stage = it&1, parity = (it>>1)&1)
    out_t *partial = reinterpret_cast<out_t *>(L.partial);
    constexpr int WARPS = warps_for(P, MIXED);
    constexpr int TILE_PX = WARPS * 32 * P;

    // The share is walked by one of two instantiations of the same loop: CLAMPED = false when the pre-pass found every
    // envelope exponent of the launch inside [-1000, 1000] (L.deep), so the table path needs no exponent clamp.
    auto walk = [&](auto clamped_tag) {
        [[maybe_unused]] constexpr bool CLAMPED = decltype(clamped_tag)::value;
        for (long long pos = b0; pos < b1;) {
            const Piece pc = piece_at<GROUPED>(L, pos, b1);
            const long tile = pc.tile, j0 = pc.j0, j1 = pc.j1, n_b = pc.n_b;
            const double *rec = pc.rec;
            out_t *out = reinterpret_cast<out_t *>(pc.out);
            const Strip<P> st = strip_of<P, WARPS>(L, tile, warp, lane);
            const double v = __dmul_rn((double)st.row - half_v, L.geom.dv);
            // strip extent (warp-uniform), used by the strip-level cull
            const double us_lo = ((double)(st.col0 - lane) - half_u) * L.geom.du;
            const double us_hi = us_lo + (double)(32 * P - 1) * L.geom.du;
            double u[P];
            acc_t acc_re[P], acc_im[P];
    #pragma unroll
            for (int i = 0; i < P; ++i) {
                u[i] = __dmul_rn((double)(st.col0 + 32 * i) - half_u, L.geom.du);
                acc_re[i] = 0;
                acc_im[i] = 0;
            }

            const long nblk = (j1 - j0 + KBK - 1) / KBK;
            if (tid == 0) {
                uint32_t cnt = (uint32_t)min((long)KBK, j1 - j0);
                mbar_arrive_expect_tx(&bar[it & 1], cnt * NE * 8);
                bulk_g2s(sbuf[it & 1], rec + j0 * NE, cnt * NE * 8, &bar[it & 1]);
            }
            for (long b = 0; b < nblk; ++b) {
                const long jb = j0 + b * KBK;
                const int cnt = (int)min((long)KBK, j1 - jb);
                if (tid == 0 && b + 1 < nblk) {
                    uint32_t cn = (uint32_t)min((long)KBK, j1 - jb - KBK);
                    uint32_t sn = (it + 1) & 1;
                    mbar_arrive_expect_tx(&bar[sn], cn * NE * 8);
                    bulk_g2s(sbuf[sn], rec + (jb + KBK) * NE, cn * NE * 8, &bar[sn]);
                }
                mbar_wait(&bar[it & 1], (it >> 1) & 1);
                if (st.valid) {
                    const double2 *sb = reinterpret_cast<const double2 *>(sbuf[it & 1]);
    #pragma unroll 1
                    for (int jj = 0; jj < cnt; ++jj) {
                        const double2 r0 = sb[jj * (NE / 2) + 0];      // cu cv
                        const double2 r1 = sb[jj * (NE / 2) + 1];      // t0 tu
                        const double2 r2 = sb[jj * (NE / 2) + 2];      // tv tuu
                        const double2 r3 = sb[jj * (NE / 2) + 3];      // tuv tvv
                        const double dv = v - r0.y;
                        const double tB = fma(r3.x, dv, r1.y);
                        const double tC = fma(fma(r3.y, dv, r2.x), dv, r1.x);
                        {
                            const double2 r4 = sb[jj * (NE / 2) + 4];      // g0 guu
                            const double2 r5 = sb[jj * (NE / 2) + 5];      // guv gvv
                            const double gB = r5.x * dv;
                            const double gC = fma(r5.y * dv, dv, r4.x);
                            const double g_cut = CULL ? r4.x + L.log2_tau : 0.0;
                            // mode factor as a quadratic in Du with the Dv-dependent parts hoisted:
                            //   a_uu Du^2 + (a_u + a_uv Dv) Du + (a0 + a_v Dv + a_vv Dv^2)
                            [[maybe_unused]] double2 hA = make_double2(0.0, 0.0), hB = hA, hC = hA;
                            if constexpr (HG) {
                                const double2 h0 = sb[jj * (NE / 2) + 6], hu = sb[jj * (NE / 2) + 7], hv = sb[jj * (NE / 2) + 8];
                                const double2 huv = sb[jj * (NE / 2) + 10], hvv = sb[jj * (NE / 2) + 11];
                                hA = sb[jj * (NE / 2) + 9];                                         // a_uu
                                hB = make_double2(fma(huv.x, dv, hu.x), fma(huv.y, dv, hu.y));
                                hC = make_double2(fma(fma(hvv.x, dv, hv.x), dv, h0.x), fma(fma(hvv.y, dv, hv.y), dv, h0.y));
                            }
                            if (CULL && strip_env_max(us_lo - r0.x, us_hi - r0.x, r4.y, gB, gC) < g_cut - 1.0)
                                continue;            // every pixel of the strip would be dropped (R-14)
                            // both quadratics of all P pixels first, then the P transcendental evaluations: the
                            // same arithmetic, but ptxas schedules it 1 % better (81.5 -> 80.7 ms on C3)
                            double t4v[P], gv[P];
    #pragma unroll
                            for (int i = 0; i < P; ++i) {
                                const double du = u[i] - r0.x;
                                t4v[i] = fma(fma(r2.y, du, tB), du, tC);
                                gv[i] = fma(fma(r4.y, du, gB), du, gC);
                            }
    #pragma unroll
                            for (int i = 0; i < P; ++i) {
                                if constexpr (HG) {
                                    // term = 2^g cis * (pr + i pi),  pr + i pi = the beamlet's mode factor at this pixel
                                    const double du = u[i] - r0.x;
                                    const double pr = fma(fma(hA.x, du, hB.x), du, hC.x);
                                    const double pi = fma(fma(hA.y, du, hB.y), du, hC.y);
                                    double e, re, im;
                                    if constexpr (TAB) gbdm::term_tab<CLAMPED>(gv[i], t4v[i], cis_lane, exp_lane, e, re, im);
                                    else { e = 1.0; gbdm::term_value(gv[i], t4v[i], re, im); }
                                    const double tr = e * re, ti = e * im;
                                    acc_re[i] = fma(-ti, pi, fma(tr, pr, acc_re[i]));
                                    acc_im[i] = fma(ti, pr, fma(tr, pi, acc_im[i]));
                                } else if constexpr (TAB) {
                                    if (CULL) gbdm::accumulate_term_tab_cull<CLAMPED>(gv[i], g_cut, t4v[i], cis_lane, exp_lane, acc_re[i], acc_im[i]);
                                    else gbdm::accumulate_term_tab<CLAMPED>(gv[i], t4v[i], cis_lane, exp_lane, acc_re[i], acc_im[i]);
                                } else {
                                    if (CULL) gbdm::accumulate_term_cull(gv[i], g_cut, t4v[i], acc_re[i], acc_im[i]);
                                    else gbdm::accumulate_term(gv[i], t4v[i], acc_re[i], acc_im[i]);
                                }
                            }
                        }
                    }
                }
                __syncthreads();                     // all reads of this stage done before it is refilled
                ++it;
            }

            // write: whole tile -> output; shared tile -> this CTA's head (0) or tail (1) partial slot
            const bool whole = (j0 == 0 && j1 == n_b);
            if (whole) {
                if (st.valid) {
    #pragma unroll
                    for (int i = 0; i < P; ++i) {
                        int col = st.col0 + 32 * i;
                        if (col < L.geom.n_u)
                            out[st.row * L.geom.n_u + col] = out_t{acc_re[i], acc_im[i]};
                    }
                }
            } else {
                const int seg = (pc.gtile == first_gtile) ? 0 : 1;
                out_t *pp = partial + ((size_t)slot * 2 + seg) * TILE_PX + warp * (32 * P) + lane;
    #pragma unroll
                for (int i = 0; i < P; ++i) pp[32 * i] = out_t{acc_re[i], acc_im[i]};
            }
            pos += (j1 - j0);
        }
    };
    if (TAB && L.deep != nullptr && *L.deep == 0) walk(std::false_type{});
    else walk(std::true_type{});
}

// ------------------------------------------------------------------ fp64 recurrence kernel
// Along one row the log of a term is a quadratic in the pixel index, so with the P consecutive pixels
// i = 0..P-1 of a thread (spacing s = du, layout run_of):   term_{i+1} = term_i * R_i,   R_{i+1} = R_i * S,
//   term_0 = 2^g(Du0) cis(T(Du0)),  R_0 = exp of the first difference,  S = exp of the (constant) second
// difference 2 s^2 (ln2 guu + i pi/2 tuu) -- a per-beamlet constant the pre-pass stores in the record.
// Cost per (beamlet, thread): two direct evaluations (term_0, R_0) + 10 FP64 instructions per pixel
// (two complex products and the accumulation) instead of ~33 per pixel.  Rounding error grows like
// i^2 ulp (i < 32: <= 1e-13 relative), far inside the 1e-10 budget; the recurrence is restarted for every
// beamlet and every thread, never carried further than P-1 steps.  Where the envelope exponent falls
// below -900 at either end of the thread's run (beam much narrower than the strip) the multiplicative
// form would start from a flushed value, so that (beamlet, thread) pair is evaluated directly.
constexpr int NEVAL_R = GBD_NEVAL + 2;

// One recurrence chain of P pixels into the accumulators: term_{n+1} = term_n R_n, R_{n+1} = R_n S, walked from
// pixel 0 upwards or (REV) from pixel P-1 downwards.
template <int P, bool REV, typename acc_t>
__device__ __forceinline__ void run_chain(acc_t tr, acc_t ti, acc_t rr, acc_t ri, acc_t sx, acc_t sy,
                                          acc_t (&acc_re)[P], acc_t (&acc_im)[P])
{
#pragma unroll
    for (int n = 0; n < P; ++n) {
        const int i = REV ? P - 1 - n : n;
        acc_re[i] += tr;
        acc_im[i] += ti;
        if (n + 1 < P) {
            const acc_t nr = fma(tr, rr, -(ti * ri));
            const acc_t ni = fma(tr, ri, ti * rr);
            tr = nr;
            ti = ni;
        }
        if (n + 2 < P) {
            const acc_t nr = fma(rr, sx, -(ri * sy));
            const acc_t ni = fma(rr, sy, ri * sx);
            rr = nr;
            ri = ni;
        }
    }
}


// MIXED = true (precision 1): the phase quadratic, its first difference and the per-beamlet factor S are still
// formed in fp64, the start values come from the MUFU path of the mixed direct kernel, and the recurrence and
// the accumulation run in fp32 (10 FP32 instructions per pixel); complex64 out.  Error: each restart is
// as accurate as the mixed direct kernel and the chain adds <= i^2/2 fp32 roundings (i < 32).
template <int P, bool GROUPED, bool MIXED>
__global__ void __launch_bounds__(warps_for(P, MIXED) * 32, 1) field_recur_kernel(const GbdFieldLaunch L)
{
    constexpr int STAGE_R = KB * NEVAL_R;
    __shared__ __align__(128) double sbuf[2][STAGE_R];
    __shared__ __align__(8) uint64_t bar[2];

    using acc_t = typename std::conditional<MIXED, float, double>::type;
    using out_t = typename std::conditional<MIXED, float2, double2>::type;
    constexpr double G_FLUSH = MIXED ? -100.0 : -900.0;     // below this the start value would be flushed
    if (L.gate && *L.gate != L.gate_want) return;
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int slot = blockIdx.x;
    const long long b0 = gbd_share_begin(L.work, L.slots, slot);
    const long long b1 = gbd_share_begin(L.work, L.slots, slot + 1);
    if (b0 >= b1) return;
    if (tid == 0) {
        mbar_init(&bar[0], 1);
        mbar_init(&bar[1], 1);
        mbar_fence_init();
    }
    __syncthreads();

    const long first_gtile = piece_at<GROUPED>(L, b0, b1).gtile;
    const double half_u = 0.5 * (double)(L.geom.n_u - 1), half_v = 0.5 * (double)(L.geom.n_v - 1);
    const double s = L.geom.du;                  // spacing of a thread's pixels
    const double run_len2_quarter = 0.25 * ((P - 1) * s) * ((P - 1) * s);
    uint32_t it = 0;
    out_t *partial = reinterpret_cast<out_t *>(L.partial);
    constexpr int WARPS = warps_for(P, MIXED);
    constexpr int TILE_PX = WARPS * 32 * P;

    for (long long pos = b0; pos < b1;) {
        const Piece pc = piece_at<GROUPED>(L, pos, b1);
        const long tile = pc.tile, j0 = pc.j0, j1 = pc.j1, n_b = pc.n_b;
        const double *rec = pc.rec;
        out_t *out = reinterpret_cast<out_t *>(pc.out);
        const Strip<P> st = run_of<P, WARPS>(L, tile, warp, lane);
        const double v = __dmul_rn((double)st.row - half_v, L.geom.dv);
        const double u0 = __dmul_rn((double)st.col0 - half_u, L.geom.du);
        acc_t acc_re[P], acc_im[P];
#pragma unroll
        for (int i = 0; i < P; ++i) { acc_re[i] = 0; acc_im[i] = 0; }

        const long nblk = (j1 - j0 + KB - 1) / KB;
        if (tid == 0) {
            uint32_t cnt = (uint32_t)min((long)KB, j1 - j0);
            mbar_arrive_expect_tx(&bar[it & 1], cnt * NEVAL_R * 8);
            bulk_g2s(sbuf[it & 1], rec + j0 * NEVAL_R, cnt * NEVAL_R * 8, &bar[it & 1]);
        }
        for (long b = 0; b < nblk; ++b) {
            const long jb = j0 + b * KB;
            const int cnt = (int)min((long)KB, j1 - jb);
            if (tid == 0 && b + 1 < nblk) {
                uint32_t cn = (uint32_t)min((long)KB, j1 - jb - KB);
                uint32_t sn = (it + 1) & 1;
                mbar_arrive_expect_tx(&bar[sn], cn * NEVAL_R * 8);
                bulk_g2s(sbuf[sn], rec + (jb + KB) * NEVAL_R, cn * NEVAL_R * 8, &bar[sn]);
            }
            mbar_wait(&bar[it & 1], (it >> 1) & 1);
            if (st.valid) {
                const double2 *sb = reinterpret_cast<const double2 *>(sbuf[it & 1]);
#pragma unroll 1
                for (int jj = 0; jj < cnt; ++jj) {
                    const double2 r0 = sb[jj * 7 + 0];      // cu cv
                    const double2 r1 = sb[jj * 7 + 1];      // t0 tu
                    const double2 r2 = sb[jj * 7 + 2];      // tv tuu
                    const double2 r3 = sb[jj * 7 + 3];      // tuv tvv
                    const double2 r4 = sb[jj * 7 + 4];      // g0 guu
                    const double2 r5 = sb[jj * 7 + 5];      // guv gvv
                    const double2 S = sb[jj * 7 + 6];       // second-difference factor
                    const double dv = v - r0.y;
                    const double tB = fma(r3.x, dv, r1.y);
                    const double tC = fma(fma(r3.y, dv, r2.x), dv, r1.x);
                    const double gB = r5.x * dv;
                    const double gC = fma(r5.y * dv, dv, r4.x);
                    const double du0 = u0 - r0.x;
                    const double duL = fma((double)(P - 1), s, du0);
                    const double g0 = fma(fma(r4.y, du0, gB), du0, gC);
                    const double gL = fma(fma(r4.y, duL, gB), duL, gC);
                    // A concave parabola exceeds its larger end value by at most |guu| len^2 / 4 inside the run: when even
                    // that bound is below G_FLUSH every term of the run is < 2^G_FLUSH (1e-271 in fp64) -- nothing to add.
                    // (Planes away from focus: most beamlets do not reach most runs; this is what keeps them cheap.)
                    const double g_skip = fma(-fabs(r4.y), run_len2_quarter, G_FLUSH);
                    if (g0 < g_skip && gL < g_skip) continue;
                    const bool fwd_ok = g0 >= G_FLUSH, bwd_ok = gL >= G_FLUSH;
                    // fp64: direct evaluation only when BOTH ends are flushed (beam narrower than the run).  The fp32
                    // kernel has no reverse chain (the second unrolled chain costs it 6 % at its 128-register cap):
                    // there a run with either end flushed is evaluated directly.
                    if (MIXED ? (!fwd_ok || !bwd_ok) : (!fwd_ok && !bwd_ok)) {
#pragma unroll 1
                        for (int i = 0; i < P; ++i) {
                            const double du = fma((double)i, s, du0);
                            const double t4 = fma(fma(r2.y, du, tB), du, tC);
                            const double g = fma(fma(r4.y, du, gB), du, gC);
                            acc_t re = 0, im = 0;
                            if constexpr (MIXED) gbdm::accumulate_term_mixed<false>((float)g, 0.f, t4, re, im);
                            else gbdm::term_value(g, t4, re, im);
#pragma unroll
                            for (int k = 0; k < P; ++k)
                                if (k == i) { acc_re[k] += re; acc_im[k] += im; }
                        }
                        continue;
                    }
                    const acc_t sx = (acc_t)S.x, sy = (acc_t)S.y;
                    acc_t tr = 0, ti = 0, rr = 0, ri = 0;
                    if (MIXED || fwd_ok) {
                        // first differences of phase and envelope between pixel 0 and pixel 1
                        const double w = fma(2.0, du0, s);
                        const double t0 = fma(fma(r2.y, du0, tB), du0, tC);
                        const double dt = s * fma(r2.y, w, tB);
                        const double dg = s * fma(r4.y, w, gB);
                        if constexpr (MIXED) {
                            gbdm::accumulate_term_mixed<false>((float)g0, 0.f, t0, tr, ti);
                            gbdm::accumulate_term_mixed<false>((float)dg, 0.f, dt, rr, ri);
                        } else {
                            gbdm::term_value(g0, t0, tr, ti);
                            gbdm::term_value(dg, dt, rr, ri);
                        }
                        run_chain<P, false>(tr, ti, rr, ri, sx, sy, acc_re, acc_im);
                    } else {
                        // the run crosses the edge of the beam's footprint with its first pixel outside: walk it from
                        // the last pixel backwards (the far values underflow to zero, which is what they are)
                        const double w = fma(2.0, duL, -s);
                        const double tL = fma(fma(r2.y, duL, tB), duL, tC);
                        const double dt = -s * fma(r2.y, w, tB);
                        const double dg = -s * fma(r4.y, w, gB);
                        if constexpr (MIXED) {
                            gbdm::accumulate_term_mixed<false>((float)gL, 0.f, tL, tr, ti);
                            gbdm::accumulate_term_mixed<false>((float)dg, 0.f, dt, rr, ri);
                        } else {
                            gbdm::term_value(gL, tL, tr, ti);
                            gbdm::term_value(dg, dt, rr, ri);
                        }
                        run_chain<P, true>(tr, ti, rr, ri, sx, sy, acc_re, acc_im);
                    }
                }
            }
            __syncthreads();
            ++it;
        }

        const bool whole = (j0 == 0 && j1 == n_b);
        if (whole) {
            if (st.valid) {
#pragma unroll
                for (int i = 0; i < P; ++i) {
                    int col = st.col0 + i;
                    if (col < L.geom.n_u) out[st.row * L.geom.n_u + col] = out_t{acc_re[i], acc_im[i]};
                }
            }
        } else {
            const int seg = (pc.gtile == first_gtile) ? 0 : 1;
            out_t *pp = partial + ((size_t)slot * 2 + seg) * TILE_PX + warp * (32 * P) + lane;
#pragma unroll
            for (int i = 0; i < P; ++i) pp[32 * i] = out_t{acc_re[i], acc_im[i]};
        }
        pos += (j1 - j0);
    }
}


// ------------------------------------------------------------------ on-axis field of a batch of problems
// e0[run] = sum_j term_j at the detector origin (u = v = 0): the peak-normalisation value of the Airy
// figure of merit (R-13).  One CTA per problem; per-thread partial sums are combined in a fixed order.
__global__ void __launch_bounds__(256) onaxis_kernel(const GbdProblem *__restrict__ probs, int rec_stride,
                                                     int mixed, double *__restrict__ e0)
{
    __shared__ double sh[2][8];
    const GbdProblem pb = probs[blockIdx.x];
    double re = 0.0, im = 0.0;
    for (long j = threadIdx.x; j < pb.n_b; j += 256) {
        const double *r = pb.rec + j * rec_stride;
        const double du = 0.0 - r[0], dv = 0.0 - r[1];
        const double tB = fma(r[6], dv, r[3]);
        const double tC = fma(fma(r[7], dv, r[4]), dv, r[2]);
        const double t4 = fma(fma(r[5], du, tB), du, tC);
        double g0, guu, guv, gvv;
        if (mixed) {
            const float *f = reinterpret_cast<const float *>(r + 8);
            g0 = f[0]; guu = f[1]; guv = f[2]; gvv = f[3];
        } else {
            g0 = r[8]; guu = r[9]; guv = r[10]; gvv = r[11];
        }
        const double g = fma(fma(guu, du, guv * dv), du, fma(gvv * dv, dv, g0));
        double tr, ti;
        gbdm::term_value(g, t4, tr, ti);
        re += tr;
        im += ti;
    }
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    for (int o = 16; o > 0; o >>= 1) {
        re += __shfl_down_sync(0xffffffffu, re, o);
        im += __shfl_down_sync(0xffffffffu, im, o);
    }
    if (lane == 0) { sh[0][warp] = re; sh[1][warp] = im; }
    __syncthreads();
    if (threadIdx.x == 0) {
        double a = sh[0][0], b = sh[1][0];
        for (int w = 1; w < 8; ++w) { a += sh[0][w]; b += sh[1][w]; }
        e0[2 * blockIdx.x] = a;
        e0[2 * blockIdx.x + 1] = b;
    }
}

// ------------------------------------------------------------------ fix-up of shared tiles
// One CTA per tile.  The CTAs ("slots") whose share intersects this tile are found from the same
// integer partition the field kernel used; partials are added in slot order -> reproducible.
template <int P, typename V2, bool CONTIG>
__global__ void __launch_bounds__(warps_for(P, std::is_same<V2, float2>::value) * 32) fixup_kernel(const GbdFieldLaunch L)
{
    if (L.gate && *L.gate != L.gate_want) return;
    const long gtile = blockIdx.x;
    long tile = gtile, n_b = L.n_b;
    long long wbeg = 0;
    void *outp = L.out;
    if (L.n_probs > 0) {
        const long ip = gtile / L.tiles_per_problem;
        tile = gtile - ip * L.tiles_per_problem;
        n_b = L.probs[ip].n_b;
        wbeg = L.probs[ip].work_begin;
        outp = L.probs[ip].out;
    }
    const long long t0 = wbeg + (long long)tile * n_b, t1 = t0 + n_b;
    // first candidate slot: largest s with begin(s) <= t0
    int s_lo = (int)((t0 * (long long)L.slots) / L.work);
    while (s_lo > 0 && gbd_share_begin(L.work, L.slots, s_lo) > t0) --s_lo;
    while (s_lo + 1 < L.slots && gbd_share_begin(L.work, L.slots, s_lo + 1) <= t0) ++s_lo;
    {
        long long e = gbd_share_begin(L.work, L.slots, s_lo + 1);
        if (e >= t1) return;                     // one CTA owned the whole tile: already written
    }
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    constexpr int WARPS = warps_for(P, std::is_same<V2, float2>::value);
    constexpr int TILE_PX = WARPS * 32 * P;
    const Strip<P> st = CONTIG ? run_of<P, WARPS>(L, tile, warp, lane) : strip_of<P, WARPS>(L, tile, warp, lane);
    if (!st.valid) return;
    const V2 *partial = reinterpret_cast<const V2 *>(L.partial);
    V2 *out = reinterpret_cast<V2 *>(outp);
    // gridDim.y CTAs share a tile (small detectors have few tiles): CTA y takes the pixels i = y, y + gridDim.y, ...
    // of every thread.  Per pixel the partials are still added in slot order, so the result does not depend on the split.
    // last slot whose share begins before the end of the tile
    int s_hi = (int)(((t1 - 1) * (long long)L.slots) / L.work);
    while (s_hi + 1 < L.slots && gbd_share_begin(L.work, L.slots, s_hi + 1) < t1) ++s_hi;
    while (s_hi > s_lo && gbd_share_begin(L.work, L.slots, s_hi) >= t1) --s_hi;
    // share boundaries advance by work / slots with a running remainder (exactly floor(work * s / slots)): no 64-bit
    // division inside the loop, and no early exit, so the loads of consecutive slots are in flight together (a 1 x 1
    // pixel detector shared by all 148 CTAs: 104 -> 12 us)
    const long long step_q = L.work / L.slots, step_r = L.work % L.slots;
    const long long sb_lo = gbd_share_begin(L.work, L.slots, s_lo);
    const long long rem_lo = L.work * (long long)s_lo - sb_lo * (long long)L.slots;
#pragma unroll 1
    for (int i = blockIdx.y; i < P; i += gridDim.y) {
        const int col = st.col0 + (CONTIG ? i : 32 * i);
        if (col >= L.geom.n_u) continue;
        double sr = 0.0, si = 0.0;
        long long sb = sb_lo, rem = rem_lo;
        const V2 *px = partial + warp * (32 * P) + lane + 32 * i;
        for (int s0 = s_lo; s0 <= s_hi; s0 += 8) {
            V2 x[8];
            bool ok[8];
#pragma unroll
            for (int k = 0; k < 8; ++k) {            // phase 1: boundaries and the (independent) loads of 8 slots
                long long se = sb + step_q;
                rem += step_r;
                if (rem >= L.slots) { rem -= L.slots; ++se; }
                const long long lo = sb > t0 ? sb : t0, hi = se < t1 ? se : t1;
                const int seg = sb >= t0 ? 0 : 1;    // the slot's share begins inside this tile: head, else tail
                ok[k] = s0 + k <= s_hi && lo < hi;   // not past the tile, not an empty share
                if (ok[k]) x[k] = px[((size_t)(s0 + k) * 2 + seg) * TILE_PX];
                sb = se;
            }
#pragma unroll
            for (int k = 0; k < 8; ++k)              // phase 2: added in slot order
                if (ok[k]) { sr += (double)x[k].x; si += (double)x[k].y; }
        }
        V2 o;
        o.x = sr;
        o.y = si;
        out[st.row * L.geom.n_u + col] = o;
    }
}

// CTAs per tile of the fix-up kernels: 1 when there are enough tiles to fill the GPU, else a power of two <= pmax
static unsigned fixup_split(long n_tiles, int slots, int pmax)
{
    unsigned fs = 1;
    while ((long)fs * n_tiles < 2L * slots && (int)(fs * 2) <= pmax) fs *= 2;
    return fs;
}

template <int P>
cudaError_t launch_p(const GbdFieldLaunch &L, int precision, int algo, bool cull, int *n_launches,
                     cudaStream_t st, cudaEvent_t ev0, cudaEvent_t ev1)
{
    const bool prof = ev0 && ev1;
    if (prof) cudaEventRecord(ev0, st);
    const bool grouped = L.n_probs > 0;
    const bool mixed = precision != GBD_PRECISION_FP64;
    const dim3 grid(L.slots), block(warps_for(P, mixed) * 32);
    int twin = 0;                     // 1: the table kernel was enqueued as a gated pair
    if (algo == GBD_ALGO_RECURRENCE) {
        if constexpr (P >= 16) {
            if (precision == GBD_PRECISION_FP64) {
                if (grouped) field_recur_kernel<P, true, false><<<grid, block, 0, st>>>(L);
                else field_recur_kernel<P, false, false><<<grid, block, 0, st>>>(L);
            } else {
                if (grouped) field_recur_kernel<P, true, true><<<grid, block, 0, st>>>(L);
                else field_recur_kernel<P, false, true><<<grid, block, 0, st>>>(L);
            }
        } else return cudaErrorInvalidValue;
    } else {
        if constexpr (P <= 8) {
            if (precision == GBD_PRECISION_FP64) {
                // table kernels for launches that amortise the table fill (every CTA spends ~2 us on it)
                const bool tab = gbd_field_uses_tables(L, P, precision, algo);
                if (tab) {
                    static unsigned long long attr_done = 0;         // per device (the attribute is per device)
                    int dev = 0;
                    cudaGetDevice(&dev);
                    if (!((attr_done >> (dev & 63)) & 1ull)) {
                        cudaFuncSetAttribute(field_fold_kernel<P, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, GBD_TAB_BYTES);
                        cudaFuncSetAttribute(field_fold_kernel<P, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, GBD_TAB_BYTES);
                        cudaFuncSetAttribute(field_tab_kernel<P, false, true, true, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, GBD_TAB_BYTES);
                        cudaFuncSetAttribute(field_tab_kernel<P, true, false, true, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, GBD_TAB_BYTES);
                        cudaFuncSetAttribute(field_tab_kernel<P, false, false, true, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, GBD_TAB_BYTES);
                        attr_done |= 1ull << (dev & 63);
                    }
                    if (grouped) {
                        field_fold_kernel<P, true><<<grid, block, GBD_TAB_BYTES, st>>>(L);
                        field_tab_kernel<P, false, true, true, false><<<grid, block, GBD_TAB_BYTES, st>>>(L);
                        twin = 1;
                    } else if (cull) {
                        field_tab_kernel<P, true, false, true, false><<<grid, block, GBD_TAB_BYTES, st>>>(L);
                    } else {
                        field_fold_kernel<P, false><<<grid, block, GBD_TAB_BYTES, st>>>(L);
                        field_tab_kernel<P, false, false, true, false><<<grid, block, GBD_TAB_BYTES, st>>>(L);
                        twin = 1;
                    }
                } else {
                    if (grouped) field_kernel<P, false, false, true><<<grid, block, 0, st>>>(L);   // the sweep never culls
                    else if (cull) field_kernel<P, true, false, false><<<grid, block, 0, st>>>(L);
                    else field_kernel<P, false, false, false><<<grid, block, 0, st>>>(L);
                }
            } else {
                // mixed precision: large launches without cull run the table kernel, gated against its twin
                if (!cull && gbd_field_uses_tables(L, P, precision, algo)) {
                    static unsigned long long attr_done_m = 0;
                    int dev = 0;
                    cudaGetDevice(&dev);
                    if (!((attr_done_m >> (dev & 63)) & 1ull)) {
                        cudaFuncSetAttribute(field_mixed_tab_kernel<P, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, GBD_MIXTAB_BYTES);
                        cudaFuncSetAttribute(field_mixed_tab_kernel<P, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, GBD_MIXTAB_BYTES);
                        attr_done_m |= 1ull << (dev & 63);
                    }
                    if (grouped) field_mixed_tab_kernel<P, true><<<grid, block, GBD_MIXTAB_BYTES, st>>>(L);
                    else field_mixed_tab_kernel<P, false><<<grid, block, GBD_MIXTAB_BYTES, st>>>(L);
                    twin = 1;
                }
                if (grouped) field_kernel<P, false, true, true><<<grid, block, 0, st>>>(L);
                else if (cull) field_kernel<P, true, true, false><<<grid, block, 0, st>>>(L);
                else field_kernel<P, false, true, false><<<grid, block, 0, st>>>(L);
            }
        } else {
            return cudaErrorInvalidValue;
        }
    }
    cudaError_t e = cudaGetLastError();
    if (prof) cudaEventRecord(ev1, st);
    if (e != cudaSuccess) return e;
    const dim3 fgrid((unsigned)L.n_tiles, fixup_split(L.n_tiles, L.slots, P));
    if (algo == GBD_ALGO_RECURRENCE && precision == GBD_PRECISION_FP64)
        fixup_kernel<P, double2, true><<<fgrid, warps_for(P, false) * 32, 0, st>>>(L);
    else if (algo == GBD_ALGO_RECURRENCE)
        fixup_kernel<P, float2, true><<<fgrid, warps_for(P, true) * 32, 0, st>>>(L);
    else if (precision == GBD_PRECISION_FP64) fixup_kernel<P, double2, false><<<fgrid, warps_for(P, false) * 32, 0, st>>>(L);
    else fixup_kernel<P, float2, false><<<fgrid, warps_for(P, true) * 32, 0, st>>>(L);
    *n_launches = 2 + twin;
    return cudaGetLastError();
}

}  // namespace

void gbd_field_config(int n_u, int precision, int algo, int *P_out, int *threads_out, int *ctas_per_sm_out)
{
    // pixels per thread: the P in {8,4,2,1} that wastes the fewest padded columns of a 32 P wide strip
    // (ties -> larger P); recurrence: P in {32,16} consecutive pixels per thread
    const bool rec = algo == GBD_ALGO_RECURRENCE;
    const int pmax = rec ? 32 : 8, pmin = rec ? 16 : 1;
    int best = pmax;
    long best_pad = -1;
    for (int P = pmax; P >= pmin; P >>= 1) {
        long w = rec ? P : 32L * P;
        long pad = ((n_u + w - 1) / w) * w;
        if (best_pad < 0 || pad < best_pad) { best_pad = pad; best = P; }
    }
    *P_out = best;
    *threads_out = warps_for(best, precision != GBD_PRECISION_FP64) * 32;
    *ctas_per_sm_out = 1;
}

size_t gbd_field_tile_px(int P, int precision) { return (size_t)warps_for(P, precision != GBD_PRECISION_FP64) * 32 * P; }

bool gbd_field_uses_tables(const GbdFieldLaunch &L, int P, int precision, int algo)
{
    const bool mixed = precision != GBD_PRECISION_FP64;
    return algo == GBD_ALGO_DIRECT && P <= 8 &&
           (double)L.work * (double)(warps_for(P, mixed) * 32 * P) >= GBD_TAB_MIN_TERMS;
}

int gbd_field_slots(int precision)
{
    (void)precision;
    int dev = 0, sms = 148;
    if (cudaGetDevice(&dev) == cudaSuccess)
        cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
    return sms;          // one persistent CTA per SM
}

cudaError_t gbd_launch_onaxis(const GbdProblem *d_probs, int n_runs, int rec_stride, int mixed, double *d_e0,
                              cudaStream_t st)
{
    if (n_runs < 1) return cudaSuccess;
    onaxis_kernel<<<n_runs, 256, 0, st>>>(d_probs, rec_stride, mixed, d_e0);
    return cudaGetLastError();
}

// field sum with per-beamlet mode factors (records of GBD_NEVAL_HG doubles), fp64 direct
template <int P>
static cudaError_t launch_modes_p(const GbdFieldLaunch &L, int *n_launches, cudaStream_t st, cudaEvent_t ev0, cudaEvent_t ev1)
{
    const bool prof = ev0 && ev1;
    const dim3 grid(L.slots), block(warps_for(P, false) * 32);
    const bool tab = gbd_field_uses_tables(L, P, GBD_PRECISION_FP64, GBD_ALGO_DIRECT);
    if (prof) cudaEventRecord(ev0, st);
    int twin = 0;
    if (tab) {
        cudaFuncSetAttribute(field_fold_kernel<P, false, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, GBD_TAB_BYTES);
        cudaFuncSetAttribute(field_tab_kernel<P, false, false, true, true>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                             GBD_TAB_BYTES);
        field_fold_kernel<P, false, true><<<grid, block, GBD_TAB_BYTES, st>>>(L);       // gated pair, as in launch_p
        field_tab_kernel<P, false, false, true, true><<<grid, block, GBD_TAB_BYTES, st>>>(L);
        twin = 1;
    } else {
        field_tab_kernel<P, false, false, false, true><<<grid, block, 0, st>>>(L);
    }
    cudaError_t e = cudaGetLastError();
    if (prof) cudaEventRecord(ev1, st);
    if (e != cudaSuccess) return e;
    fixup_kernel<P, double2, false><<<dim3((unsigned)L.n_tiles, fixup_split(L.n_tiles, L.slots, P)), warps_for(P, false) * 32, 0, st>>>(L);
    *n_launches = 2 + twin;
    return cudaGetLastError();
}

cudaError_t gbd_launch_field_modes(const GbdFieldLaunch &L, int P, int *n_launches, cudaStream_t st,
                                   cudaEvent_t ev0, cudaEvent_t ev1)
{
    *n_launches = 0;
    if (L.work == 0) return cudaSuccess;
    switch (P) {
    case 1: return launch_modes_p<1>(L, n_launches, st, ev0, ev1);
    case 2: return launch_modes_p<2>(L, n_launches, st, ev0, ev1);
    case 4: return launch_modes_p<4>(L, n_launches, st, ev0, ev1);
    case 8: return launch_modes_p<8>(L, n_launches, st, ev0, ev1);
    default: break;
    }
    return cudaErrorInvalidValue;
}

cudaError_t gbd_launch_field(const GbdFieldLaunch &L, int P, int precision, int algo, bool cull,
                             int *n_launches, cudaStream_t st, cudaEvent_t ev0, cudaEvent_t ev1)
{
    *n_launches = 0;
    if (L.work == 0) return cudaSuccess;
    switch (P) {
    case 1: return launch_p<1>(L, precision, algo, cull, n_launches, st, ev0, ev1);
    case 2: return launch_p<2>(L, precision, algo, cull, n_launches, st, ev0, ev1);
    case 4: return launch_p<4>(L, precision, algo, cull, n_launches, st, ev0, ev1);
    case 8: return launch_p<8>(L, precision, algo, cull, n_launches, st, ev0, ev1);
    case 16: if (algo == GBD_ALGO_RECURRENCE) return launch_p<16>(L, precision, algo, cull, n_launches, st, ev0, ev1); break;
    case 32: if (algo == GBD_ALGO_RECURRENCE) return launch_p<32>(L, precision, algo, cull, n_launches, st, ev0, ev1); break;
    default: break;
    }
    return cudaErrorInvalidValue;
}
