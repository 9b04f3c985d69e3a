// gbd_sep.cu -- the field sum for beamlets WITHOUT a cross term (algo 2; fp64, or fp32 tables and updates): when Q_xy + Q_yx = 0 for every
// beamlet (any rotationally symmetric system on axis: all of C0-C3) the term factorises,
//     term_j(u, v) = F_j(u) * G_j(v),
//     F_j(u) = 2^(g0 + guu Du^2) cis(pi/2 (t0 + tu Du + tuu Du^2)),   G_j(v) = 2^(gvv Dv^2) cis(pi/2 (tv Dv + tvv Dv^2)),
// and a pixel tile only needs the TU + TV edge values of each beamlet: the sum over beamlets becomes a chain of
// complex rank-1 updates, 4 DFMA per (beamlet, pixel) -- the same sum as P:33 Eq. 3 / P:153-157 Eq. 20, evaluated
// in a different order.  Whether the factorisation applies is decided on the device by the pre-pass (a gate word in
// the workspace): this kernel runs when the gate is clear, the general recurrence kernel when it is set.
//
//   tile    = TU x TV = 128 x 64 pixels (fp32: 128 x 128, k < 16), one 256-thread CTA: warp w owns rows w + 8k (k < 8), lane l columns
//             l + 32i (i < 4), so the G values a warp needs are warp-uniform (broadcast loads);
//   work    = n_tiles * n_b beamlet-tile units in 148 equal contiguous shares (stream-K, as in gbd_field.cu);
//   records = 16 doubles per beamlet (evaluation record + the second-difference factors S_u, S_v), streamed by
//             1-D bulk async copies in blocks of 128, double buffered;
//   phase A = for a sub-block of 16 beamlets the edge tables F[16][128], G[16][64] are filled in shared memory by
//             24 lanes of every warp, each running one 16-value along-edge recurrence (two direct evaluations +
//             8 FP64 instructions per value); the 16 steps of the NEXT sub-block's recurrence are interleaved
//             with the 16 beamlet iterations of phase B, so their latency chain is hidden;
//   phase B = every thread: per beamlet 4 + 8 LDS.128, 32 complex multiply-adds = 128 DFMA.
#include <type_traits>

#include "gbd_common.cuh"
#include "gbd_math.cuh"
#include "gbd_tile.cuh"

namespace {

constexpr int SEP_THREADS = 256;                        // 8 warps: warp w owns rows w + 8k, lane l columns l + 32i
constexpr int KS = 16;                                  // beamlets per table sub-block
constexpr int NREC_S = 16;                              // doubles per record
constexpr int RUN = 16;                                 // values per phase-A thread
static_assert(KS == RUN, "one recurrence step is interleaved with every beamlet of phase B");

// Tile and per-thread pixels.  fp64: 128 x 64, 4 x 8 pixels per thread (64 accumulators = 128 registers).
// fp32: 128 x 128, 4 x 16 pixels per thread -- the same 128 accumulator registers, half the table loads and
// integer work per multiply-add.
template <typename T> struct SepCfg {
    static constexpr int TU = 128, TV = 64, PU = 4, PV = 8;
};
template <> struct SepCfg<float> {
    static constexpr int TU = 128, TV = 128, PU = 4, PV = 16;
};

// T = double: precision 0.  T = float: precision 1 -- records and the start values of every edge recurrence as in
// the mixed direct kernel (fp64 phase -> fixed-point turn -> MUFU), tables, recurrence and rank-1 updates in fp32.
template <typename T> struct vec2 { using type = double2; };
template <> struct vec2<float> { using type = float2; };

template <typename T>
struct SepSmem {
    typename vec2<T>::type F[2][KS][SepCfg<T>::TU];
    typename vec2<T>::type G[2][KS][SepCfg<T>::TV];
    double rec[2][KB * NREC_S];
    uint64_t bar[2];
    // reach[buf][beamlet]: 1 when the beamlet has a live column run AND a live row run (a run is live when it holds
    // a value above the flush threshold); otherwise it cannot reach the tile and phase B skips it.
    unsigned char reach[2][KS];
};

template <typename T>
__device__ __forceinline__ void term_of(double g, double t4, T &re, T &im);
template <>
__device__ __forceinline__ void term_of<double>(double g, double t4, double &re, double &im)
{
    gbdm::term_value(g, t4, re, im);
}
template <>
__device__ __forceinline__ void term_of<float>(double g, double t4, float &re, float &im)
{
    re = 0.f;
    im = 0.f;
    gbdm::accumulate_term_mixed<false>((float)g, 0.f, t4, re, im);
}

// Table slot of edge value p (0..TU-1 / 0..TV-1): values come in chunks of 16 (one recurrence run each); inside
// chunk c the value k sits at (k + c) mod 16, so the 12 runs a warp stores at the same step k hit different
// banks while a chunk stays one contiguous 256-byte range for the loads of phase B.
__device__ __forceinline__ int slot_of(int p) { return (p & ~15) | ((p + (p >> 4)) & 15); }

// One along-edge recurrence in flight: values 2^g(D) cis(pi/2 t(D)) at D = D0 + k h, k = 0..RUN-1, with
// t(D) = c0 + c1 D + c2 D^2, g(D) = e0 + e2 D^2:   term_{k+1} = term_k R_k,  R_{k+1} = R_k S.
template <typename T>
struct EdgeRun {
    T tr, ti, rr, ri, sx, sy;
    typename vec2<T>::type *chunk;      // the 16-slot chunk this run fills
    int rot, sgn;        // value number k of the walk goes to slot (rot + sgn k) mod 16: rot = chunk index (slot
                         // rotation), sgn = +1; a run walked from its last value backwards: rot = chunk index + 15, sgn = -1
    bool live;           // false: nothing to step (idle lane, or the values were written directly)
};

template <typename T>
__device__ __forceinline__ bool edge_begin(EdgeRun<T> &e, bool on, double D0, double h, double c0, double c1, double c2,
                                           double e0, double e2, double sx, double sy,
                                           typename vec2<T>::type *chunk, int rot)
{
    using T2 = typename vec2<T>::type;
    constexpr double G_FLUSH = std::is_same<T, float>::value ? -100.0 : -900.0;
    e.live = false;
    e.chunk = chunk;
    e.rot = rot;
    e.sx = (T)sx;
    e.sy = (T)sy;
    e.tr = e.ti = e.rr = e.ri = 0;
    e.sgn = 1;
    if (!on) return false;
    const double DL = fma((double)(RUN - 1), h, D0);
    const double g0 = fma(e2 * D0, D0, e0), gL = fma(e2 * DL, DL, e0);
    // a concave parabola exceeds its larger end value by at most |e2| len^2 / 4: below the flush threshold
    // everywhere -> the run is dead (zeros; the caller records it)
    const double g_skip = fma(-fabs(e2), 0.25 * ((RUN - 1) * h) * ((RUN - 1) * h), G_FLUSH);
    if (g0 < g_skip && gL < g_skip) {
#pragma unroll
        for (int k = 0; k < RUN; ++k) chunk[k] = T2{0, 0};
        return false;
    }
    const bool fwd_ok = g0 >= G_FLUSH, bwd_ok = gL >= G_FLUSH;
    if (!fwd_ok && !bwd_ok) {                    // beam narrower than the run: evaluate directly
#pragma unroll 1
        for (int k = 0; k < RUN; ++k) {
            const double D = fma((double)k, h, D0);
            T re, im;
            term_of<T>(fma(e2 * D, D, e0), fma(fma(c2, D, c1), D, c0), re, im);
            chunk[(k + rot) & 15] = T2{re, im};
        }
        return true;
    }
    // start from the end whose value is representable and walk towards the other (a run crossing the edge of the
    // beam's footprint is walked from inside out; the far values underflow to zero, which is what they are)
    const bool rev = !fwd_ok;
    if (rev) { e.rot = rot + RUN - 1; e.sgn = -1; }
    const double DS = rev ? DL : D0, hs = rev ? -h : h;
    const double w = fma(2.0, DS, hs);
    term_of<T>(rev ? gL : g0, fma(fma(c2, DS, c1), DS, c0), e.tr, e.ti);
    term_of<T>(hs * (e2 * w), hs * fma(c2, w, c1), e.rr, e.ri);
    e.live = true;
    return true;
}

template <typename T>
__device__ __forceinline__ void edge_step(EdgeRun<T> &e, int k)
{
    using T2 = typename vec2<T>::type;
    if (e.live) e.chunk[(e.rot + e.sgn * k) & 15] = T2{e.tr, e.ti};
    const T nr = fma(e.tr, e.rr, -(e.ti * e.ri)), ni = fma(e.tr, e.ri, e.ti * e.rr);
    e.tr = nr; e.ti = ni;
    const T mr = fma(e.rr, e.sx, -(e.ri * e.sy)), mi = fma(e.rr, e.sy, e.ri * e.sx);
    e.rr = mr; e.ri = mi;
}

template <typename T, bool GROUPED>
__global__ void __launch_bounds__(SEP_THREADS, 1) field_sep_kernel(const GbdFieldLaunch L)
{
    using T2 = typename vec2<T>::type;
    constexpr int TU = SepCfg<T>::TU, TV = SepCfg<T>::TV, PU = SepCfg<T>::PU, PV = SepCfg<T>::PV;
    constexpr int TILE_PX_S = TU * TV;
    constexpr int RUNS_PER_BEAMLET = (TU + TV) / RUN;            // 8 along u, 4 (8) along v
    constexpr int A_LANES = KS * RUNS_PER_BEAMLET / (SEP_THREADS / 32);   // lanes of every warp with a phase-A run
    static_assert(A_LANES <= 32 && A_LANES * (SEP_THREADS / 32) == KS * RUNS_PER_BEAMLET, "phase-A roles");
    static_assert(TU == 32 * PU && TV == (SEP_THREADS / 32) * PV, "thread tile");
    extern __shared__ __align__(128) unsigned char smem_raw[];
    SepSmem<T> &sm = *reinterpret_cast<SepSmem<T> *>(smem_raw);
    if (L.gate && *L.gate != L.gate_want) return;

    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int slot = blockIdx.x;
    const long long b0 = gbd_share_begin(L.work, L.slots, slot);
    const long long b1 = gbd_share_begin(L.work, L.slots, slot + 1);
    if (b0 >= b1) return;
    if (tid == 0) {
        mbar_init(&sm.bar[0], 1);
        mbar_init(&sm.bar[1], 1);
        mbar_fence_init();
    }
    __syncthreads();

    const long first_gtile = piece_at<GROUPED>(L, b0, b1).gtile;
    const double half_u = 0.5 * (double)(L.geom.n_u - 1), half_v = 0.5 * (double)(L.geom.n_v - 1);
    const int tiles_u = L.strips_per_row;
    uint32_t it = 0;
    T2 *partial = reinterpret_cast<T2 *>(L.partial);
    // phase-A role: the first A_LANES lanes of every warp run one recurrence: beamlet a_j of the sub-block, run
    // a_run (0..7: 16 columns each, 8..: 16 rows each)
    const bool a_on = lane < A_LANES;
    const int a_idx = warp * A_LANES + (a_on ? lane : 0);
    const int a_j = a_idx / RUNS_PER_BEAMLET, a_run = a_idx - a_j * RUNS_PER_BEAMLET;
    const bool a_is_f = a_run < TU / RUN;
    const int a_rot = a_is_f ? a_run : a_run - TU / RUN;
    const double a_h = a_is_f ? L.geom.du : L.geom.dv;
    // phase-B table slots of this thread
    int fslot[PU], gslot[PV];
#pragma unroll
    for (int i = 0; i < PU; ++i) fslot[i] = slot_of(lane + 32 * i);
#pragma unroll
    for (int k = 0; k < PV; ++k) gslot[k] = slot_of(warp + 8 * k);

    for (long long pos = b0; pos < b1;) {
        const Piece pc = piece_at<GROUPED>(L, pos, b1);
        const long tile = pc.tile, j0 = pc.j0, j1 = pc.j1, n_b = pc.n_b;
        const double *rec = pc.rec;
        T2 *out = reinterpret_cast<T2 *>(pc.out);
        const long tile_v = tile / tiles_u;
        const int col0 = (int)(tile - tile_v * tiles_u) * TU;
        const long row0 = tile_v * TV;
        const double a_x0 = a_is_f ? __dmul_rn((double)(col0 + a_rot * RUN) - half_u, L.geom.du)
                                   : __dmul_rn((double)(row0 + a_rot * RUN) - half_v, L.geom.dv);
        T acc_re[PV][PU], acc_im[PV][PU];
#pragma unroll
        for (int k = 0; k < PV; ++k)
#pragma unroll
            for (int i = 0; i < PU; ++i) { acc_re[k][i] = 0; acc_im[k][i] = 0; }

        // start the recurrence of this thread's run for sub-block `sub` of record stage `rb` into table `buf`
        auto begin_run = [&](EdgeRun<T> &e, const double *rb, int sub, int ns, int buf) {
            const double *r = rb + (sub * KS + (a_j < ns ? a_j : 0)) * NREC_S;
            const bool on = a_on && a_j < ns;
            T2 *chunk = a_is_f ? &sm.F[buf][a_j][a_rot * RUN] : &sm.G[buf][a_j][a_rot * RUN];
            const bool alive = edge_begin<T>(e, on, a_x0 - r[a_is_f ? 0 : 1], a_h, a_is_f ? r[2] : 0.0,
                                             r[a_is_f ? 3 : 4], r[a_is_f ? 5 : 7], a_is_f ? r[8] : 0.0,
                                             r[a_is_f ? 9 : 11], r[a_is_f ? 12 : 14], r[a_is_f ? 13 : 15], chunk, a_rot);
            // the RUNS_PER_BEAMLET runs of one beamlet sit in consecutive lanes of one warp: combine by ballot
            const unsigned live = __ballot_sync(0xffffffffu, alive && on);
            const int grp = (lane / RUNS_PER_BEAMLET) * RUNS_PER_BEAMLET;         // first lane of this beamlet's runs
            const unsigned runs = (live >> grp) & ((1u << RUNS_PER_BEAMLET) - 1u);
            const unsigned fmask = (1u << (TU / RUN)) - 1u;
            if (on && a_run == 0) sm.reach[buf][a_j] = ((runs & fmask) != 0u && (runs & ~fmask) != 0u) ? 1 : 0;
        };
        // 16-bit mask of the beamlets of table `buf` that reach this tile (read once per sub-block, after the barrier)
        auto reach_mask = [&](int buf) {
            const uint4 r4 = *reinterpret_cast<const uint4 *>(&sm.reach[buf][0]);
            unsigned m = 0;
            const unsigned wds[4] = { r4.x, r4.y, r4.z, r4.w };
#pragma unroll
            for (int q = 0; q < 4; ++q)
#pragma unroll
                for (int b2 = 0; b2 < 4; ++b2) m |= ((wds[q] >> (8 * b2)) & 1u) << (4 * q + b2);
            return m;
        };

        const long nblk = (j1 - j0 + KB - 1) / KB;
        if (tid == 0) {
            uint32_t cnt = (uint32_t)min((long)KB, j1 - j0);
            mbar_arrive_expect_tx(&sm.bar[it & 1], cnt * NREC_S * 8);
            bulk_g2s(sm.rec[it & 1], rec + j0 * NREC_S, cnt * NREC_S * 8, &sm.bar[it & 1]);
        }
        uint32_t tb = 0;                         // table buffer counter
        for (long b = 0; b < nblk; ++b) {
            const long jb = j0 + b * KB;
            const int cnt = (int)min((long)KB, j1 - jb);
            if (tid == 0 && b + 1 < nblk) {
                uint32_t cn = (uint32_t)min((long)KB, j1 - jb - KB);
                uint32_t sn = (it + 1) & 1;
                mbar_arrive_expect_tx(&sm.bar[sn], cn * NREC_S * 8);
                bulk_g2s(sm.rec[sn], rec + (jb + KB) * NREC_S, cn * NREC_S * 8, &sm.bar[sn]);
            }
            mbar_wait(&sm.bar[it & 1], (it >> 1) & 1);
            const double *rb = sm.rec[it & 1];
            const int nsub = (cnt + KS - 1) / KS;
            EdgeRun<T> er;
            // tables of the first sub-block of this record stage: nothing to overlap them with
            begin_run(er, rb, 0, min(KS, cnt), tb & 1);
#pragma unroll
            for (int k = 0; k < RUN; ++k) edge_step(er, k);
            __syncthreads();
            for (int sub = 0; sub < nsub; ++sub, ++tb) {
                const int ns = min(KS, cnt - sub * KS);
                const int buf = tb & 1;
                const bool next = sub + 1 < nsub;            // then ns == KS == RUN
                if (next) begin_run(er, rb, sub + 1, min(KS, cnt - (sub + 1) * KS), buf ^ 1);
                else er.live = false;
                // beamlets that do not reach the tile are skipped in the fp64 loop (planes away from focus: 13.8 -> 6.8 ms
                // on a defocused C3 plane for 2.6 % at focus); the fp32 loop is issue-bound and the test costs it 6 %, so
                // there dead runs just contribute their zeros
                const unsigned rmask = std::is_same<T, double>::value ? reach_mask(buf) : 0xffffu;
                // phase B (rank-1 updates from table `buf`) with one step of the next tables' recurrence each
                if constexpr (std::is_same<T, double>::value) {
#pragma unroll 2
                    for (int jj = 0; jj < ns; ++jj) {
                        if (!((rmask >> jj) & 1u)) {         // block-uniform: this beamlet does not reach the tile
                            edge_step(er, jj);
                            continue;
                        }
                        T2 f[PU], g[PV];
#pragma unroll
                        for (int i = 0; i < PU; ++i) f[i] = sm.F[buf][jj][fslot[i]];
#pragma unroll
                        for (int k = 0; k < PV; ++k) g[k] = sm.G[buf][jj][gslot[k]];
                        edge_step(er, jj);
#pragma unroll
                        for (int k = 0; k < PV; ++k) {
                            const T ngi = -g[k].y;
#pragma unroll
                            for (int i = 0; i < PU; ++i) {
                                acc_re[k][i] = fma(g[k].x, f[i].x, acc_re[k][i]);
                                acc_im[k][i] = fma(g[k].x, f[i].y, acc_im[k][i]);
                            }
#pragma unroll
                            for (int i = 0; i < PU; ++i) {
                                acc_re[k][i] = fma(ngi, f[i].y, acc_re[k][i]);
                                acc_im[k][i] = fma(g[k].y, f[i].x, acc_im[k][i]);
                            }
                        }
                    }
                } else {
                    // fp32: the table loads are software-pipelined -- the G value of row-update k+1 and, half-way,
                    // the F values of the next beamlet are requested while row-update k runs (6.49 -> 6.16 ms on C3;
                    // the fp64 loop is FP64-pipe bound and loses 3 % with the same interleaving)
                    T2 f_next[PU], g_cur;
#pragma unroll
                    for (int i = 0; i < PU; ++i) f_next[i] = sm.F[buf][0][fslot[i]];
                    g_cur = sm.G[buf][0][gslot[0]];
#pragma unroll 2
                    for (int jj = 0; jj < ns; ++jj) {
                        T2 f[PU];
#pragma unroll
                        for (int i = 0; i < PU; ++i) f[i] = f_next[i];
                        const int jn = min(jj + 1, ns - 1);      // last beamlet: a harmless re-load
                        edge_step(er, jj);
#pragma unroll
                        for (int k = 0; k < PV; ++k) {
                            const T2 g = g_cur;
                            g_cur = (k + 1 < PV) ? sm.G[buf][jj][gslot[k + 1]] : sm.G[buf][jn][gslot[0]];
                            if (k == PV / 2) {
#pragma unroll
                                for (int i = 0; i < PU; ++i) f_next[i] = sm.F[buf][jn][fslot[i]];
                            }
                            const T ngi = -g.y;
#pragma unroll
                            for (int i = 0; i < PU; ++i) {
                                acc_re[k][i] = fma(g.x, f[i].x, acc_re[k][i]);
                                acc_im[k][i] = fma(g.x, f[i].y, acc_im[k][i]);
                            }
#pragma unroll
                            for (int i = 0; i < PU; ++i) {
                                acc_re[k][i] = fma(ngi, f[i].y, acc_re[k][i]);
                                acc_im[k][i] = fma(g.y, f[i].x, acc_im[k][i]);
                            }
                        }
                    }
                }
                __syncthreads();                 // table buf^1 complete, all reads of table buf done
            }
            ++it;
        }

        const bool whole = (j0 == 0 && j1 == n_b);
        if (whole) {
#pragma unroll
            for (int k = 0; k < PV; ++k) {
                const long row = row0 + warp + 8 * k;
#pragma unroll
                for (int i = 0; i < PU; ++i) {
                    const int col = col0 + lane + 32 * i;
                    if (row < L.geom.n_v && col < L.geom.n_u)
                        out[row * L.geom.n_u + col] = T2{acc_re[k][i], acc_im[k][i]};
                }
            }
        } else {
            const int seg = (pc.gtile == first_gtile) ? 0 : 1;
            T2 *pp = partial + ((size_t)slot * 2 + seg) * TILE_PX_S + tid;
#pragma unroll
            for (int k = 0; k < PV; ++k)
#pragma unroll
                for (int i = 0; i < PU; ++i) pp[(k * PU + i) * SEP_THREADS] = T2{acc_re[k][i], acc_im[k][i]};
        }
        pos += (j1 - j0);
    }
}

// One CTA per tile: adds the partial sums of the CTAs that shared it, in slot order (bitwise reproducible).
template <typename T>
__global__ void __launch_bounds__(SEP_THREADS) fixup_sep_kernel(const GbdFieldLaunch L)
{
    constexpr int TU = SepCfg<T>::TU, TV = SepCfg<T>::TV, PU = SepCfg<T>::PU, PV = SepCfg<T>::PV;
    constexpr int TILE_PX_S = TU * TV;
    if (L.gate && *L.gate != L.gate_want) return;
    long tile = blockIdx.x, n_b = L.n_b;
    long long wbeg = 0;
    void *outp = L.out;
    if (L.n_probs > 0) {
        const long ip = tile / L.tiles_per_problem;
        tile -= ip * L.tiles_per_problem;
        n_b = L.probs[ip].n_b;
        wbeg = L.probs[ip].work_begin;
        outp = L.probs[ip].out;
    }
    const long long t0 = wbeg + (long long)tile * n_b, t1 = t0 + n_b;
    int s_lo = (int)((t0 * (long long)L.slots) / L.work);
    while (s_lo > 0 && gbd_share_begin(L.work, L.slots, s_lo) > t0) --s_lo;
    while (s_lo + 1 < L.slots && gbd_share_begin(L.work, L.slots, s_lo + 1) <= t0) ++s_lo;
    if (gbd_share_begin(L.work, L.slots, s_lo + 1) >= t1) return;      // one CTA owned the whole tile
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    using T2 = typename vec2<T>::type;
    const T2 *partial = reinterpret_cast<const T2 *>(L.partial);
    const int tiles_u = L.strips_per_row;
    const long tile_v = tile / tiles_u;
    const int col0 = (int)(tile - tile_v * tiles_u) * TU;
    const long row0 = tile_v * TV;
    T2 *out = reinterpret_cast<T2 *>(outp);
    // gridDim.y CTAs share a tile (small detectors have few tiles): CTA y takes the pixels q = y, y + gridDim.y, ... of
    // every thread; per pixel the partials are still added in slot order.
#pragma unroll 1
    for (int q = blockIdx.y; q < PV * PU; q += gridDim.y) {
        const int k = q / PU, i = q - k * PU;
        const long row = row0 + warp + 8 * k;
        const int col = col0 + lane + 32 * i;
        if (row >= L.geom.n_v || col >= L.geom.n_u) continue;
        double sr = 0.0, si = 0.0;
        for (int s = s_lo; s < L.slots; ++s) {
            const long long sb = gbd_share_begin(L.work, L.slots, s), se = gbd_share_begin(L.work, L.slots, s + 1);
            if (sb >= t1) break;
            const long long lo = sb > t0 ? sb : t0, hi = se < t1 ? se : t1;
            if (lo >= hi) continue;
            const int seg = sb >= t0 ? 0 : 1;
            const T2 x = partial[((size_t)s * 2 + seg) * TILE_PX_S + tid + q * SEP_THREADS];
            sr += (double)x.x;
            si += (double)x.y;
        }
        out[row * L.geom.n_u + col] = T2{(T)sr, (T)si};
    }
}

}  // namespace

void gbd_sep_geometry(int n_u, int n_v, int precision, int *tiles_u, long *n_tiles)
{
    const int tu = precision == GBD_PRECISION_FP64 ? SepCfg<double>::TU : SepCfg<float>::TU;
    const int tv = precision == GBD_PRECISION_FP64 ? SepCfg<double>::TV : SepCfg<float>::TV;
    *tiles_u = (n_u + tu - 1) / tu;
    *n_tiles = (long)*tiles_u * ((n_v + tv - 1) / tv);
}

template <typename T, bool GROUPED>
static cudaError_t launch_sep(const GbdFieldLaunch &L, cudaStream_t st, cudaEvent_t ev0, cudaEvent_t ev1)
{
    cudaError_t e = cudaFuncSetAttribute(field_sep_kernel<T, GROUPED>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                         (int)sizeof(SepSmem<T>));     // per device, cheap
    if (e != cudaSuccess) return e;
    const bool prof = ev0 && ev1;
    if (prof) cudaEventRecord(ev0, st);
    field_sep_kernel<T, GROUPED><<<L.slots, SEP_THREADS, sizeof(SepSmem<T>), st>>>(L);
    e = cudaGetLastError();
    if (prof) cudaEventRecord(ev1, st);
    if (e != cudaSuccess) return e;
    unsigned fs = 1;                         // CTAs per tile: fill the GPU when the detector has few tiles
    while ((long)fs * L.n_tiles < 2L * L.slots && fs < 32) fs *= 2;
    fixup_sep_kernel<T><<<dim3((unsigned)L.n_tiles, fs), SEP_THREADS, 0, st>>>(L);
    return cudaGetLastError();
}

// slots: one CTA per SM for both precisions (two co-resident fp32 CTAs are capped at 128 registers, which makes the
// compiler recompute the table addresses in the loop: 7.5 ms against 6.5 ms on C3)
int gbd_sep_slots(int precision, int sms) { (void)precision; return sms; }

cudaError_t gbd_launch_field_sep(const GbdFieldLaunch &L, int precision, int *n_launches, cudaStream_t st,
                                 cudaEvent_t ev0, cudaEvent_t ev1)
{
    *n_launches = 0;
    if (L.work == 0) return cudaSuccess;
    const bool grouped = L.n_probs > 0;
    cudaError_t e;
    if (precision == GBD_PRECISION_FP64)
        e = grouped ? launch_sep<double, true>(L, st, ev0, ev1) : launch_sep<double, false>(L, st, ev0, ev1);
    else
        e = grouped ? launch_sep<float, true>(L, st, ev0, ev1) : launch_sep<float, false>(L, st, ev0, ev1);
    if (e == cudaSuccess) *n_launches = 2;
    return e;
}
