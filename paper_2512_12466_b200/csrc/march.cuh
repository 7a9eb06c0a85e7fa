// The ray loop on the device: scheduler, emit, march+deposit+filter+split (DESIGN.md rows a4-a8), field
// preparation and finalise (a9).
//
// One launch marches a batch of rays that all sit on the SAME HEALPix level (the pool is one stack per
// level), so the split radius, the pixel width and the expected number of cells per ray are uniform
// across a launch.  Each ray is marched to its end: tau >= tau_max (filter), box exit
// (BASELINE.json configs; reading R20) or the split criterion Eq. 4, in which case the
// four children are pushed on the stack of level+1.
//
// Kernel shape (sm_100a, latency- and issue-bound rather than HBM-bound, see profiles/): persistent warps.
// A warp claims chunks of 32 rays, sets them up at full width and parks them in a shared-memory queue; a
// lane whose ray ended pops the next one, so ray-length tails do not idle lanes.  Per cell the work is split
// into a geometry stage (DDA, Eq. 5-8 geometry, the two absorber gathers) that runs TWO cells ahead of the
// physics stage (absorption, deposits), through three segment descriptors in registers.  The ray's read-only
// direction and 1/d live in shared memory.  The grids are padded by one halo cell holding -inf: leaving the
// box is "the absorber I just loaded is -inf", a neighbour outside the box is never eligible, and no cell
// coordinates are tracked.
//
// Everything that steers control flow follows DESIGN.md's DEC list literally; this translation unit is
// compiled with -fmad=false.
#pragma once
#include "healpix.cuh"
#include "state.cuh"

namespace nyxrt {

constexpr int MARCH_THREADS = 128;
constexpr int MARCH_WARPS = MARCH_THREADS / 32;
constexpr int MARCH_MIN_BLOCKS = 4;      // 16 warps per SM at <= 128 registers, no spills (checked with -Xptxas -v); a fifth
                                         // block (96 registers, 132 KB of shared memory) measured 6 % slower
#ifndef MARCH_SEG_ROUND
#define MARCH_SEG_ROUND 21                // cells a lane marches between two retire / refill passes (15 and 30: within 0.7 %)
#endif
constexpr int MARCH_CARVEOUT = 40;       // preferred shared-memory carve-out [% of 228 KB]: 4 blocks x 21 KB

// ---------------------------------------------------------------------------------------------------
// Scheduler: one thread decides what the next emit + march launches do.
//   1. deepest level holding a full batch; else
//   2. if sources remain, top level 0 up with 12 rays per source, then 1. again; else
//   3. the shallowest non-empty level (drain).
// With caps of 2B (level 0) and 5B + slab slack (deeper levels) no stack can overflow.
__device__ __forceinline__ void sched_decide(LoopState *ls, DevStats *ds, const RayPool &pool, int nlev) {
    ls->emit_n = 0;
    ls->batch = 0;
    ls->fetch = 0;
    if (ls->overflow) ls->done = 1;                          // a pool overflow ends the loop: EOVERFLOW, never garbage
    if (ls->done) return;
    const long long B = ls->batch_rays;
    int pick = -1;
    for (int l = nlev - 1; l >= 0; --l)
        if (ls->count[l] >= B) { pick = l; break; }
    if (pick < 0 && ls->src_next < ls->n_cat) {
        long long room = (pool.cap[0] - ls->count[0]) / 12;
        long long k = ls->n_cat - ls->src_next;
        if (k > room) k = room;
        if (k > 0) {
            ls->emit_src = ls->src_next;
            ls->emit_n = k;
            ls->emit_slot = pool.off[0] + ls->count[0];
            ls->count[0] += 12 * k;
            ls->src_next += k;
        }
        if (ls->count[0] >= B) pick = 0;
    }
    if (pick < 0) {
        if (ls->src_next < ls->n_cat) pick = 0;          // cannot happen with cap[0] >= 2B; stay safe
        else
            for (int l = 0; l < nlev; ++l)
                if (ls->count[l] > 0) { pick = l; break; }
    }
    if (pick < 0 || ls->count[pick] == 0) {
        if (ls->emit_n == 0) ls->done = 1;
        return;
    }
    long long total = 0;
    for (int l = 0; l < nlev; ++l) total += ls->count[l];
    if ((unsigned long long)total > ls->peak_pool) ls->peak_pool = (unsigned long long)total;
    long long b = ls->count[pick] < B ? ls->count[pick] : B;
    ls->count[pick] -= b;
    ls->level = pick;
    ls->begin = pool.off[pick] + ls->count[pick];
    ls->batch = b;
    ls->seg_round = pick < 2 ? 3 : MARCH_SEG_ROUND;
    ls->iterations += 1;
    ds->spawned[pick] += (unsigned long long)b;          // every slot is popped exactly once (holes subtracted later)
}

// `cond`: the handle of the CUDA-graph WHILE node that wraps sched -> emit -> march when the loop runs as one graph
// launch (nyxrt.cu); the loop goes on while it is non-zero.  use_cond = 0: launched from the host loop.
__global__ void sched_kernel(LoopState *ls, DevStats *ds, RayPool pool, int nlev, cudaGraphConditionalHandle cond,
                             int use_cond) {
    if (threadIdx.x != 0 || blockIdx.x != 0) return;
    sched_decide(ls, ds, pool, nlev);
    if (use_cond) cudaGraphSetConditional(cond, ls->done ? 0u : 1u);
}

// ---------------------------------------------------------------------------------------------------
// Emit (PAPER.md:111, 203 spawn_rays): 12 level-0 rays per catalogue source, L/12 each.
// Source sharding: shard `rank` of `world` emits the catalogue sources rank, rank + world, ...
__global__ void emit_kernel(const LoopState *ls, RayPool pool, const double *cat_L, int rank, int world) {
    const long long n = ls->emit_n * 12;
    const long long src0 = ls->emit_src, slot0 = ls->emit_slot;
    for (long long r = (long long)blockIdx.x * blockDim.x + threadIdx.x; r < n;
         r += (long long)gridDim.x * blockDim.x) {
        const long long a = (src0 + r / 12) * world + rank;
        const uint32_t pix = (uint32_t)(r % 12);
        pool.key[slot0 + r] = ray_key((uint32_t)a, 0, pix);
        pool.s[slot0 + r] = 0.0;
        pool.tau[slot0 + r] = 0.0;
        pool.N[slot0 + r] = cat_L[a] / 12.0;
    }
}

// ---------------------------------------------------------------------------------------------------
// pm = e^-x - 1 (minus the absorbed fraction) and left = e^-x for x >= 0 (not DEC: the tolerance is 1e-9,
// DESIGN.md "Tolerances").  One branch-free routine for thin and thick cells (they sit side by side in every warp):
// x = k ln2 + r with |r| <= ln2/2 (k = 0 for a thin cell); e^-r - 1 = u + u^2 q(u), u = -r, by its Taylor series through u^11
// (remainder < 2e-14 relative); left = 2^-k (1 + p), pm = 2^-k p + (2^-k - 1): e^-x - 1 keeps full relative
// accuracy where 1 - exp(-x) would not.  Coefficients sit in constant memory so that they are
// operands, not re-materialised immediates.
__constant__ double EXPC[10] = {1.0 / 39916800.0, 1.0 / 3628800.0, 1.0 / 362880.0, 1.0 / 40320.0, 1.0 / 5040.0,
                                1.0 / 720.0,      1.0 / 120.0,     1.0 / 24.0,     1.0 / 6.0,     0.5};

__device__ __forceinline__ void absorb_fraction(double x, double &pm, double &left) {
    const double xc = x < 700.0 ? x : 700.0;                     // e^-700 ~ 1e-304: nothing is left either way
    const double MAGIC = 6755399441055744.0;                     // 1.5 * 2^52: round to nearest integer
    const double kd_m = fma(xc, 1.4426950408889634, MAGIC);
    const int k = __double2loint(kd_m);                          // 0 .. 1010
    const double kd = kd_m - MAGIC;
    double r = fma(kd, -6.93147180369123816490e-01, xc);         // ln2 hi
    r = fma(kd, -1.90821492927058770002e-10, r);                 // ln2 lo
    const double u = -r;
    double q = EXPC[0];
#pragma unroll
    for (int i = 1; i < 10; ++i) q = fma(q, u, EXPC[i]);
    const double p = fma(u * u, q, u);                           // e^u - 1
    const double sc = __hiloint2double((1023 - k) << 20, 0);     // 2^-k
    left = fma(sc, p, sc);
    pm = fma(sc, p, sc - 1.0);
}

// a / b to a few ulp without the IEEE slow path (not DEC: only scales a deposit); b is a positive normal
// number.  The hardware seed is good to ~2^-20; one Newton step squares that and the residual correction of
// the quotient squares it again, so the result is rounding-limited.  (The correction is needed: the
// neighbour's share is 1 - f_c = 1/2 - a/b, which cancels when D_edge is close to L_pix/2, and a cell may
// receive nothing but such shares.)
__device__ __forceinline__ double div_fast(double a, double b) {
    double y;
    asm("rcp.approx.ftz.f64 %0, %1;" : "=d"(y) : "d"(b));
    const double e = fma(-b, y, 1.0);
    y = fma(y, e, y);
    const double qv = a * y;
    return fma(fma(-b, qv, a), y, qv);
}

// +-1.0 and +-0.5 with the sign of x (x = 1/d: the direction of travel along one axis)
__device__ __forceinline__ double signed_one(double x) {
    return __hiloint2double((__double2hiint(x) & 0x80000000) | 0x3ff00000, 0);
}
__device__ __forceinline__ double signed_half(double x) {
    return __hiloint2double((__double2hiint(x) & 0x80000000) | 0x3fe00000, 0);
}

enum { OUT_NONE = 0, OUT_SPLIT = 1, OUT_KILL_TAU = 2, OUT_EXIT = 3, OUT_KILL_LMAX = 4 };

// per-thread scratch that is touched only when a ray is born or retires (kept out of registers)
template <bool ON, typename V, int N>
struct OptArray { V v[N]; };
template <typename V, int N>
struct OptArray<false, V, N> {};          // not needed by this instantiation: takes no shared memory

template <int LUT>
struct ThreadScratch {
    unsigned long long key[MARCH_THREADS];
    double esc[MARCH_THREADS], res[MARCH_THREADS];
    OptArray<LUT != 0, double, MARCH_THREADS> w;   // spectrum table: the ray's share of its source's photons (constant)
    double d[3][MARCH_THREADS];          // the lane's ray: HEALPix direction and 1/d (read-only while it marches;
    double inv[3][MARCH_THREADS];        // kept out of the register file so that 5 blocks fit an SM)
};

// warp-uniform bookkeeping that only the retire path touches
struct WarpScratch {
    long long slab_pos[MARCH_WARPS], slab_end[MARCH_WARPS];       // child slots reserved on the stack of level+1
    unsigned int n_split[MARCH_WARPS], n_ktau[MARCH_WARPS], n_exit[MARCH_WARPS], n_klmax[MARCH_WARPS], n_hole[MARCH_WARPS];
};

// Frequency-integrated flux (Sec. 2.2): absorbed fraction Q(tau_0) of a ray's share between the
// source and threshold optical depth tau_0, tabulated on the binary buckets of tau_0 (2^m nodes per octave from
// 2^e_lo to 2^e_hi, linear in tau_0 inside a bucket; linear from 0 below the table, constant above it: R38).
// Bit operations and one fma: the same number on the host oracle and here.
__device__ __forceinline__ double lut_q(const MarchArgs &A, double tau) {
    if (!(tau > 0.0)) return 0.0;
    if (tau < A.lut_t_lo) return A.lut_q_first * (tau * A.lut_inv_t_lo);
    if (tau >= A.lut_t_hi) return A.lut_q_last;
    const long long bits = __double_as_longlong(tau);
    const long long k = (bits >> A.lut_fb) - A.lut_k0;
    const double frac = (double)(bits & A.lut_fmask) * A.lut_fscale;
    const double q0 = __ldg(A.lut_q + k), q1 = __ldg(A.lut_q + k + 1);
    return fma(frac, q1 - q0, q0);
}

// The separate table for thin segments (PAPER.md:267 footnote 3; R40): T = dQ/dtau_0 on the nodes of Q, the same
// interpolation, constant below the first node and above the last.
__device__ __forceinline__ double lut_t(const MarchArgs &A, double tau) {
    if (!(tau >= A.lut_t_lo)) return A.lut_t_first;
    if (tau >= A.lut_t_hi) return A.lut_t_last;
    const long long bits = __double_as_longlong(tau);
    const long long k = (bits >> A.lut_fb) - A.lut_k0;
    const double frac = (double)(bits & A.lut_fmask) * A.lut_fscale;
    const double t0 = __ldg(A.lut_t + k), t1 = __ldg(A.lut_t + k + 1);
    return fma(frac, t1 - t0, t0);
}

// Both tables through one gather pair (LUT == 2): `thin` picks T (and its edge rule) or Q; the value is lut_t's or
// lut_q's, bit for bit.  Lanes of a warp that disagree on `thin` then still share one lookup instead of running
// the two routines one after the other.
__device__ __forceinline__ double lut_qt(const MarchArgs &A, double x, bool thin) {
    if (!(x >= A.lut_t_lo)) return thin ? A.lut_t_first : (x > 0.0 ? A.lut_q_first * (x * A.lut_inv_t_lo) : 0.0);
    if (x >= A.lut_t_hi) return thin ? A.lut_t_last : A.lut_q_last;
    const long long bits = __double_as_longlong(x);
    const long long k = (bits >> A.lut_fb) - A.lut_k0;
    const double frac = (double)(bits & A.lut_fmask) * A.lut_fscale;
    const double *__restrict__ tab = thin ? A.lut_t : A.lut_q;
    const double v0 = __ldg(tab + k), v1 = __ldg(tab + k + 1);
    return fma(frac, v1 - v0, v0);
}

// One ray-cell segment, described by the geometry stage and consumed by the physics stage one iteration
// later (so that its two absorber gathers have a whole iteration to arrive).
template <typename IDX>
struct SegDesc {
    double a_c, a_n;      // absorber of the cell (sign = Eq. 7-8 flag, -inf = outside the box) and of the neighbour
    double ds, fc;        // length; f_c = 1/2 + D_edge / L_pix of Eq. 5 / 7
    IDX c, cq;            // cell and neighbour across the nearest face (cq == c: no neighbour deposit)
    int split;            // 1: the cell's entry distance meets Eq. 4: the ray splits here instead of marching;
                          // 2 (periodic box): the entry distance is no longer below sqrt(3) L_box: the ray ends
};

// Rays of the current chunk that passed their birth tests, initialised at full warp width and parked until
// a lane falls idle (one queue of FETCH_CHUNK = 32 entries per warp; positions are never stored).
static_assert(FETCH_CHUNK == 32, "one chunk = one ray per lane");
template <typename IDX, bool PER>
struct RayQueue {
    unsigned long long key[MARCH_WARPS][32];
    double s[MARCH_WARPS][32], tau[MARCH_WARPS][32], N[MARCH_WARPS][32];
    double d0[MARCH_WARPS][32], d1[MARCH_WARPS][32], d2[MARCH_WARPS][32];           // HEALPix direction
    double inv0[MARCH_WARPS][32], inv1[MARCH_WARPS][32], inv2[MARCH_WARPS][32];     // 1/d (-inf where d = 0)
    IDX c[MARCH_WARPS][32];                                                          // start cell
    OptArray<PER, unsigned long long, MARCH_WARPS * 32> cnt;                         // periodic box: steps to each face
};

// Periodic box: the ray's cell index stays inside the box.  cnt packs, 21 bits per
// axis, the number of steps the ray can still take along that axis before it crosses the box face;
// the step that crosses lands on the opposite side instead (c moves by (1 - n) strides).
constexpr int WRAP_BITS = 21;
constexpr unsigned long long WRAP_MASK = (1ull << WRAP_BITS) - 1ull;

// GEOM: 0 no correction, 1 Eq. 5 only, 3 Eq. 5-6 / 7-8 (neighbour deposit; flags live in the field), 4 squared
// PER: periodic box: cells wrap, rays end at s >= sqrt(3) L_box, the halo holds the wrapped
// images of the opposite faces (neighbour reads) and deposits into it are folded back by finalise.
// LUT = 2: the Q table plus the table for thin segments (R40-R42): a segment with dtau < tau_thin absorbs
// w dtau T(tau + dtau / 2); N is the photon count the ray carries, counted down segment by segment, as in the
// monochromatic kernel, and the share w is recomputed from the source's luminosity when the ray is popped.
// LUT = 1: absorbed photons from the spectrum table, w [Q(tau + dtau) - Q(tau)], instead of the monochromatic
// N (1 - e^-dtau); the lane's N register then holds Q(tau) and the pool's N the share w.
template <int GEOM, typename IDX, bool PER, int LUT>
__global__ void __launch_bounds__(MARCH_THREADS, MARCH_MIN_BLOCKS) march_kernel(const __grid_constant__ MarchArgs A) {
    __shared__ ThreadScratch<LUT> T;
    __shared__ RayQueue<IDX, PER> Q;
    __shared__ WarpScratch W;
    const int wid = threadIdx.x >> 5;
    const LoopState *ls = A.ls;
    const long long batch = ls->batch;
    if (batch == 0) return;
    const int level = ls->level;
    const int seg_round = ls->seg_round;
    const long long begin = ls->begin;
    const int lane = threadIdx.x & 31;
    const unsigned lt = (1u << lane) - 1u;
    const double r2s = A.r2_split[level], Kl = A.K[level];
    const double Kh = 0.5 * A.K[level];
    const double tau_max = A.tau_max, sdx = A.sdx;
    const double s_max = A.s_max;
    const IDX sy = (IDX)A.px, sz = (IDX)A.pxy;
    const double *__restrict__ absorber = A.absorber;
    double *__restrict__ acc = A.acc;

    T.esc[threadIdx.x] = 0.0;
    T.res[threadIdx.x] = 0.0;
    unsigned int n_seg = 0, n_zero = 0, n_nbr = 0;
    double lost = 0.0;
    if (lane == 0) {
        W.slab_pos[wid] = W.slab_end[wid] = 0;
        W.n_split[wid] = W.n_ktau[wid] = W.n_exit[wid] = W.n_klmax[wid] = W.n_hole[wid] = 0u;
    }
    __syncwarp();

    // warp-uniform bookkeeping
    int qhead = 0, qn = 0;                          // the warp's parked rays: entries [qhead, qhead+qn)
    bool exhausted = false;

    // per-lane ray state.  The DDA (s, od, sx, c) runs TWO CELLS AHEAD of the physics: it describes the next
    // cell to be traversed, while two of SA / SB / SC hold the segments whose absorber loads are in flight.
    bool has = false;
    double s = 0.0, tau = 0.0, N = 0.0;
    double q_tau = -1.0;               // LUT == 2: Q(tau) left by the last thick segment (Q >= 0; -1: look it up)
    double od0 = 0, od1 = 0, od2 = 0, sx0 = 0, sx1 = 0, sx2 = 0;
    IDX c = 0;                                     // cell (padded linear index)
    unsigned long long cnt = 0;                    // periodic box: steps left to the faces (3 x 21 bits)
    SegDesc<IDX> SA, SB, SC;
    SA.split = SB.split = SC.split = 0;

    // G stage: describe the cell the DDA stands in (everything here is geometry: no loaded value is needed),
    // issue its absorber loads, and advance the DDA to the next cell.  A cell that meets the split criterion
    // (Eq. 4, tested on the entry distance s) is only flagged: the DDA stays put, so that the children
    // inherit s, and only the cell's own absorber is fetched (the box-exit test comes first).
    auto describe = [&](SegDesc<IDX> &D) {
        D.c = c;
        D.a_c = __ldg(absorber + c);
        int flag = s * s > r2s ? 1 : 0;
        if (PER && !(s < s_max)) flag = 2;                                        // RAY_FLTR, PAPER.md:174 (before split)
        D.split = flag;
        D.cq = c;
        D.a_n = 0.0;
        if (flag) return;                                                         // rare: once per ray at most
        double s_exit = sx0; int ax = 0;
        if (sx1 < s_exit) { s_exit = sx1; ax = 1; }
        if (sx2 < s_exit) { s_exit = sx2; ax = 2; }                               // first minimum, order x, y, z
        double ds = s_exit - s;
        if (!(ds > 0.0)) ds = 0.0;
        D.ds = ds;
        D.fc = 1.0;
        if (GEOM != 0) {
            const double s_m = fma(0.5, ds, s);                                   // = s + 0.5 ds (0.5 ds is exact)
            double m0 = fma(s_m, T.d[0][threadIdx.x], 0.5) - od0;
            double m1 = fma(s_m, T.d[1][threadIdx.x], 0.5) - od1;
            double m2 = fma(s_m, T.d[2][threadIdx.x], 0.5) - od2;
            // nearest face, first minimum in the order x-, x+, y-, y+, z-, z+ (ties inside an axis go to the
            // minus side, ties between axes to the earlier axis: the same choice as six sequential tests)
            const double t0 = 1.0 - m0, t1 = 1.0 - m1, t2 = 1.0 - m2;
            double h0 = m0; IDX f0 = (IDX)-1;
            if (t0 < h0) { h0 = t0; f0 = (IDX)1; }
            double h1 = m1; IDX f1 = -sy;
            if (t1 < h1) { h1 = t1; f1 = sy; }
            double h2 = m2; IDX f2 = -sz;
            if (t2 < h2) { h2 = t2; f2 = sz; }
            double de = h0; IDX off = f0;
            if (h1 < de) { de = h1; off = f1; }
            if (h2 < de) { de = h2; off = f2; }
            if (de < 0.0) {
                // rounding put the midpoint a hair outside the cell: redo with the clamp to [0, 1] of the
                // DEC list (rare; when every m is inside [0, 1] the clamp changes nothing)
                m0 = m0 < 0.0 ? 0.0 : (m0 > 1.0 ? 1.0 : m0);
                m1 = m1 < 0.0 ? 0.0 : (m1 > 1.0 ? 1.0 : m1);
                m2 = m2 < 0.0 ? 0.0 : (m2 > 1.0 ? 1.0 : m2);
                de = m0; off = (IDX)-1;
                double t = 1.0 - m0; if (t < de) { de = t; off = (IDX)1; }
                if (m1 < de) { de = m1; off = -sy; }
                t = 1.0 - m1; if (t < de) { de = t; off = sy; }
                if (m2 < de) { de = m2; off = -sz; }
                t = 1.0 - m2; if (t < de) { de = t; off = sz; }
            }
            if (de < s_m * Kh && ds > 0.0) {                            // D_edge < L_pix / 2  (Eq. 5 / 7)
                D.cq = c + off;                                                   // cq != c marks "eligible"
                if (GEOM == 3) D.a_n = __ldg(absorber + D.cq);
            }
            // f_c = 1/2 + D_edge / L_pix, L_pix = s_m sqrt(Omega) (R22): geometry too; used only when the
            // neighbour takes its share (then s_m > 0)
            D.fc = 0.5 + div_fast(de, s_m * Kl);
        }
        // advance one cell (DEC: s = s_exit; s_a = ((o_a + [d_a > 0]) - 0.5) / d_a)
        s = s_exit;
        const double iv = T.inv[ax][threadIdx.x];
        const double one = signed_one(iv), half = signed_half(iv);
        if (ax == 0) { od0 += one; sx0 = (od0 + half) * iv; }
        if (ax == 1) { od1 += one; sx1 = (od1 + half) * iv; }
        if (ax == 2) { od2 += one; sx2 = (od2 + half) * iv; }
        const IDX ustp = ax == 0 ? (IDX)1 : (ax == 1 ? sy : sz);
        const IDX stp = __double2hiint(iv) < 0 ? -ustp : ustp;                  // 1/d < 0: the ray moves down the axis
        if (PER) {
            const int sh = WRAP_BITS * ax;
            const int n_ax = ax == 0 ? A.nx : (ax == 1 ? A.ny : A.nz);
            if (((cnt >> sh) & WRAP_MASK) == 0ull) {                              // crosses the face: wrap around
                c += stp - stp * (IDX)n_ax;
                cnt += (unsigned long long)(n_ax - 1) << sh;
            } else {
                c += stp;
                cnt -= 1ull << sh;
            }
        } else {
            c += stp;
        }
    };

    // P stage: the tests in the oracle's order (box exit, filter, split), then the segment's absorption and
    // its deposit (Eq. 1-2, 5-8).  Returns the ray's outcome.
    auto physics = [&](const SegDesc<IDX> &D) -> int {
        int outcome;
        if (PER) {
            outcome = tau >= tau_max ? OUT_KILL_TAU : (D.split == 2 ? OUT_EXIT : (D.split ? OUT_SPLIT : OUT_NONE));
        } else {
            const bool f_exit = __double2hiint(D.a_c) == (int)0xfff00000;
            outcome = f_exit ? OUT_EXIT : (tau >= tau_max ? OUT_KILL_TAU : (D.split ? OUT_SPLIT : OUT_NONE));
        }
        if (outcome == OUT_NONE) {
            if (D.ds > 0.0) {
                ++n_seg;
                const double dtau = (fabs(D.a_c) * sdx) * D.ds;
                double pm, left, dN;
                if constexpr (LUT == 2) {
                    // thin: dtau T(tau + dtau/2); thick: Q(tau + dtau) - Q(tau), where Q(tau) is the previous thick
                    // segment's Q(tau + dtau) -- `tau` is that very double, so the carried value has the bits a second
                    // lookup would return; it is looked up only after a thin segment or a pop
                    const bool thin = dtau < A.tau_thin;
                    const double v = lut_qt(A, thin ? tau + 0.5 * dtau : tau + dtau, thin);
                    double q_a = q_tau;
                    if (!thin && q_a < 0.0) q_a = lut_q(A, tau);
                    const double frac = thin ? dtau * v : v - q_a;
                    q_tau = thin ? -1.0 : v;
                    dN = T.w.v[threadIdx.x] * frac;
                    left = N - dN;
                    pm = 0.0;
                } else if constexpr (LUT == 1) {
                    left = lut_q(A, tau + dtau);                                  // Q at the end of the segment
                    dN = T.w.v[threadIdx.x] * (left - N);
                } else {
                    absorb_fraction(dtau, pm, left);
                    dN = N * (-pm);
                }
                if (dN > 0.0) {
                    double fc = 1.0;
                    if (GEOM == 3) {
                        if (D.a_n > 0.0) {                                        // in the box, absorber > 0, n_H >= n_th
                            fc = D.fc;
                            ++n_nbr;
                            atomicAdd(acc + D.cq, (1.0 - fc) * dN);
                        }
                    } else if (GEOM == 1 || GEOM == 4) {
                        if (D.cq != D.c) { fc = D.fc; if (GEOM == 4) fc = fc * fc; }
                        lost += (1.0 - fc) * dN;
                    }
                    atomicAdd(acc + D.c, fc * dN);
                }
                N = LUT != 0 ? left : N * left;
                tau = tau + dtau;
            } else {
                ++n_zero;
            }
        }
        return outcome;
    };

    // retire rays whose outcome is known (all lanes call it; outcome NONE = nothing to do)
    // rN: photons the ray still carries (budget); rW: what its children share (= rN, or the share w with a table)
    auto retire = [&](int outcome, double rs, double rtau, double rN, double rW, unsigned long long rkey) {
        const unsigned m_any = __ballot_sync(0xffffffffu, outcome != OUT_NONE);
        if (m_any == 0) return;
        const unsigned m_split = __ballot_sync(0xffffffffu, outcome == OUT_SPLIT);
        const unsigned m_ktau = __ballot_sync(0xffffffffu, outcome == OUT_KILL_TAU);
        const unsigned m_exit = __ballot_sync(0xffffffffu, outcome == OUT_EXIT);
        const unsigned m_klmax = __ballot_sync(0xffffffffu, outcome == OUT_KILL_LMAX);
        if (lane == 0) {
            W.n_split[wid] += __popc(m_split); W.n_ktau[wid] += __popc(m_ktau); W.n_exit[wid] += __popc(m_exit);
            W.n_klmax[wid] += __popc(m_klmax);
        }
        if (outcome == OUT_EXIT) T.esc[threadIdx.x] += rN;
        else if (outcome == OUT_KILL_TAU || outcome == OUT_KILL_LMAX) T.res[threadIdx.x] += rN;
        if (m_split) {
            // children go to the warp's slab on the stack of level+1; when the slab cannot hold them all, the
            // first `rem` slots (a multiple of 4) finish the old slab and the rest start a new one: no slot is
            // wasted, so B marched rays push at most 4B children (+ one partly used slab per warp per launch)
            const int need = 4 * __popc(m_split);
            long long slab_pos = W.slab_pos[wid], slab_end = W.slab_end[wid];
            __syncwarp();
            const long long rem = slab_end - slab_pos;
            long long base = 0;
            if (need > rem) {
                if (lane == 0) base = (long long)atomicAdd((unsigned long long *)&A.ls->count[level + 1],
                                                           (unsigned long long)CHILD_SLAB);
                base = __shfl_sync(0xffffffffu, base, 0);
                if (base + CHILD_SLAB > A.pool.cap[level + 1]) {
                    if (lane == 0) A.ls->overflow = 1;
                    for (long long h = slab_pos + lane; h < slab_end; h += 32) A.pool.key[A.pool.off[level + 1] + h] = KEY_HOLE;
                    if (lane == 0) W.slab_pos[wid] = W.slab_end[wid] = 0;
                    __syncwarp();
                    return;
                }
            }
            if (outcome == OUT_SPLIT) {
                const long long lo = 4 * __popc(m_split & lt);
                const long long w = A.pool.off[level + 1] + (lo < rem ? slab_pos + lo : base + (lo - rem));
                const uint32_t src = key_src(rkey), p4 = 4u * key_pix(rkey);
                const double Nc = rW * 0.25;                                     // L shared evenly
#pragma unroll
                for (int k = 0; k < 4; ++k) {
                    A.pool.key[w + k] = ray_key(src, level + 1, p4 + k);
                    A.pool.s[w + k] = rs;
                    A.pool.tau[w + k] = rtau;
                    A.pool.N[w + k] = Nc;
                }
            }
            if (need > rem) { slab_pos = base + (need - rem); slab_end = base + CHILD_SLAB; }
            else slab_pos += need;
            if (lane == 0) { W.slab_pos[wid] = slab_pos; W.slab_end[wid] = slab_end; }
            __syncwarp();
        }
    };

    for (;;) {
        // ---- stage: when the warp's queue is empty, ALL 32 lanes initialise the next chunk of the batch ----
        // (HEALPix direction, 1/d, start cell, birth tests), whatever rays they are marching: the expensive
        // set-up runs at full width, rays that end at birth (outside the box, depleted, split at once) are
        // retired on the spot, the others are parked in shared memory until a lane falls idle.
        if (qn == 0 && !exhausted) {
            unsigned long long f = 0;
            if (lane == 0) f = atomicAdd((unsigned long long *)&A.ls->fetch, (unsigned long long)FETCH_CHUNK);
            f = __shfl_sync(0xffffffffu, f, 0);
            if ((long long)f >= batch) { exhausted = true; continue; }
            const bool mine = (long long)f + lane < batch;
            const long long r = begin + (long long)f + lane;
            int outcome = OUT_NONE;
            unsigned long long ikey = KEY_HOLE;
            if (mine) ikey = A.pool.key[r];
            const bool real = ikey != KEY_HOLE;
            const unsigned m_hole = __ballot_sync(0xffffffffu, mine && !real);
            if (lane == 0) W.n_hole[wid] += __popc(m_hole);
            double ts = 0.0, ttau = 0.0, tN = 0.0, e0 = 0.0, e1 = 0.0, e2 = 0.0, i0 = 0.0, i1 = 0.0, i2 = 0.0;
            IDX tc = 0;
            unsigned long long tcnt = 0;
            bool park = false;
            if (real) {
                ts = A.pool.s[r];
                ttau = A.pool.tau[r];
                tN = A.pool.N[r];
                const int4 sc = A.cat_cell[key_src(ikey)];
                pix2dir(level, key_pix(ikey), e0, e1, e2);
                // O4: start-of-life cell, source-relative (source at its cell centre)
                double q, o0, o1, o2;
                q = fma(ts, e0, 0.5); o0 = floor(q); if (q == o0 && e0 < 0.0) o0 -= 1.0;
                q = fma(ts, e1, 0.5); o1 = floor(q); if (q == o1 && e1 < 0.0) o1 -= 1.0;
                q = fma(ts, e2, 0.5); o2 = floor(q); if (q == o2 && e2 < 0.0) o2 -= 1.0;
                i0 = (e0 == 0.0) ? -CUDART_INF : 1.0 / e0;                     // with od + (-0.5): s_x = +inf
                i1 = (e1 == 0.0) ? -CUDART_INF : 1.0 / e1;
                i2 = (e2 == 0.0) ? -CUDART_INF : 1.0 / e2;
                long long ci = sc.x + (long long)o0, cj = sc.y + (long long)o1, ck = sc.z + (long long)o2;
                if (PER) {
                    ci %= A.nx; if (ci < 0) ci += A.nx;
                    cj %= A.ny; if (cj < 0) cj += A.ny;
                    ck %= A.nz; if (ck < 0) ck += A.nz;
                    tcnt = (unsigned long long)(e0 > 0.0 ? A.nx - 1 - ci : ci) |
                           ((unsigned long long)(e1 > 0.0 ? A.ny - 1 - cj : cj) << WRAP_BITS) |
                           ((unsigned long long)(e2 > 0.0 ? A.nz - 1 - ck : ck) << (2 * WRAP_BITS));
                }
                if (!PER && (ci < 0 || ci >= A.nx || cj < 0 || cj >= A.ny || ck < 0 || ck >= A.nz)) outcome = OUT_EXIT;
                else if (ttau >= tau_max) outcome = OUT_KILL_TAU;
                else if (level >= A.level_max) outcome = OUT_KILL_LMAX;
                else if (PER && !(ts < s_max)) outcome = OUT_EXIT;
                else if (ts * ts > r2s) outcome = OUT_SPLIT;
                else {
                    tc = (IDX)(((ck + 1) * A.pxy) + (cj + 1) * A.px + (ci + 1));
                    park = true;
                }
            }
            const unsigned m_park = __ballot_sync(0xffffffffu, park);
            if (park) {
                const int e = __popc(m_park & lt);
                Q.key[wid][e] = ikey;
                Q.s[wid][e] = ts; Q.tau[wid][e] = ttau; Q.N[wid][e] = tN;
                Q.d0[wid][e] = e0; Q.d1[wid][e] = e1; Q.d2[wid][e] = e2;
                Q.inv0[wid][e] = i0; Q.inv1[wid][e] = i1; Q.inv2[wid][e] = i2;
                Q.c[wid][e] = tc;
                if constexpr (PER) Q.cnt.v[wid * 32 + e] = tcnt;
            }
            qhead = 0;
            qn = __popc(m_park);
            __syncwarp();
            retire(outcome, ts, ttau, (LUT == 1 && outcome != OUT_NONE) ? tN * (1.0 - lut_q(A, ttau)) : tN, tN, ikey);
            continue;
        }
        // ---- pop: idle lanes take parked rays ------------------------------------------------------------
        const unsigned m_idle = __ballot_sync(0xffffffffu, !has);
        if (m_idle != 0 && qn > 0) {
            const int n_idle = __popc(m_idle);
            const int take = n_idle < qn ? n_idle : qn;
            const int rank = __popc(m_idle & lt);
            if (!has && rank < take) {
                const int e = qhead + rank;
                T.key[threadIdx.x] = Q.key[wid][e];
                s = Q.s[wid][e]; tau = Q.tau[wid][e]; N = Q.N[wid][e];
                q_tau = -1.0;
                if constexpr (LUT == 1) { T.w.v[threadIdx.x] = N; N = lut_q(A, tau); }
                if constexpr (LUT == 2)                                           // the share L / (12 4^l)
                    T.w.v[threadIdx.x] = A.cat_L[key_src(Q.key[wid][e])] / (12.0 * (double)(1ll << (2 * level)));
                const double d0 = Q.d0[wid][e], d1 = Q.d1[wid][e], d2 = Q.d2[wid][e];
                const double inv0 = Q.inv0[wid][e], inv1 = Q.inv1[wid][e], inv2 = Q.inv2[wid][e];
                T.d[0][threadIdx.x] = d0; T.d[1][threadIdx.x] = d1; T.d[2][threadIdx.x] = d2;
                T.inv[0][threadIdx.x] = inv0; T.inv[1][threadIdx.x] = inv1; T.inv[2][threadIdx.x] = inv2;
                c = Q.c[wid][e];
                if constexpr (PER) cnt = Q.cnt.v[wid * 32 + e];
                double q;
                q = fma(s, d0, 0.5); od0 = floor(q); if (q == od0 && d0 < 0.0) od0 -= 1.0;
                q = fma(s, d1, 0.5); od1 = floor(q); if (q == od1 && d1 < 0.0) od1 -= 1.0;
                q = fma(s, d2, 0.5); od2 = floor(q); if (q == od2 && d2 < 0.0) od2 -= 1.0;
                sx0 = (od0 + signed_half(inv0)) * inv0;                        // ((o + [d > 0]) - 0.5) / d
                sx1 = (od1 + signed_half(inv1)) * inv1;
                sx2 = (od2 + signed_half(inv2)) * inv2;
                has = true;
                // pending segment = a null one (zero length, no deposit): the first pair of the march
                // describes the real first cell; the null segment's zero-length tally is taken back here
                SA.a_c = 0.0; SA.a_n = 0.0; SA.ds = 0.0; SA.fc = 1.0; SA.c = c; SA.cq = c; SA.split = 0;
                SB = SA;
                n_zero -= 1u;
                n_zero -= 1u;
            }
            qhead += take;
            qn -= take;
            __syncwarp();
        }
        if (__ballot_sync(0xffffffffu, has) == 0) {
            if (exhausted && qn == 0) break;                                      // nothing staged, nothing in flight
            continue;
        }
        // ---- march: seg_round/3 triples of cells per lane, then retire / refill ------------------------
        // Software pipeline: while the physics of one segment runs, the geometry stage has already issued
        // the loads of the next two (a gather has two iterations to arrive).
        int outcome = OUT_NONE;
        for (int it = 0; it < seg_round; it += 3) {
            if (has && outcome == OUT_NONE) {
                // SA, SB pending (in that order) on entry and on exit.  A flagged segment (split / travel limit)
                // stops the DDA: the descriptors behind it are not described, only marked, and never processed.
                if (!SB.split) describe(SC); else SC.split = SB.split;
                outcome = physics(SA);
                if (outcome == OUT_NONE) {
                    if (!SC.split) describe(SA); else SA.split = SC.split;
                    outcome = physics(SB);
                    if (outcome == OUT_NONE) {
                        if (!SA.split) describe(SB); else SB.split = SA.split;
                        outcome = physics(SC);
                    }
                }
            }
        }
        if constexpr (LUT == 1) {
            const double w = T.w.v[threadIdx.x];
            retire(outcome, s, tau, w * (1.0 - N), w, outcome == OUT_SPLIT ? T.key[threadIdx.x] : 0ull);
        } else {
            retire(outcome, s, tau, N, N, outcome == OUT_SPLIT ? T.key[threadIdx.x] : 0ull);
        }
        if (outcome != OUT_NONE) has = false;
    }
    // pad the unused tail of the last child slab
    __syncwarp();
    for (long long h = W.slab_pos[wid] + lane; h < W.slab_end[wid]; h += 32) A.pool.key[A.pool.off[level + 1] + h] = KEY_HOLE;

    // flush per-thread / per-warp tallies
    unsigned long long seg64 = n_seg, zero64 = n_zero, nbr64 = n_nbr;
    double esc = T.esc[threadIdx.x], res = T.res[threadIdx.x];
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) {
        seg64 += __shfl_xor_sync(0xffffffffu, seg64, o);
        zero64 += __shfl_xor_sync(0xffffffffu, zero64, o);
        nbr64 += __shfl_xor_sync(0xffffffffu, nbr64, o);
        esc += __shfl_xor_sync(0xffffffffu, esc, o);
        res += __shfl_xor_sync(0xffffffffu, res, o);
        lost += __shfl_xor_sync(0xffffffffu, lost, o);
    }
    if (lane == 0) {
        DevStats *ds = A.ds;
        if (seg64) atomicAdd(&ds->segments, seg64);
        if (zero64) atomicAdd(&ds->zero_len, zero64);
        if (nbr64) atomicAdd(&ds->nbr_deposits, nbr64);
        if (W.n_split[wid]) atomicAdd(&ds->split[level], (unsigned long long)W.n_split[wid]);
        if (W.n_ktau[wid]) atomicAdd(&ds->killed_tau[level], (unsigned long long)W.n_ktau[wid]);
        if (W.n_exit[wid]) atomicAdd(&ds->exited[level], (unsigned long long)W.n_exit[wid]);
        if (W.n_klmax[wid]) atomicAdd(&ds->killed_lmax[level], (unsigned long long)W.n_klmax[wid]);
        if (W.n_hole[wid]) atomicAdd(&ds->holes[level], (unsigned long long)W.n_hole[wid]);
        if (esc != 0.0) atomicAdd(&ds->escaped, esc);
        if (res != 0.0) atomicAdd(&ds->residual, res);
        if (lost != 0.0) atomicAdd(&ds->lost, lost);
    }
}

// ---------------------------------------------------------------------------------------------------
// Field preparation (set_fields): absorber a = n_H x_HI in fp64 (reading R1) on the PADDED
// grid, with the sign bit carrying Eq. 7-8's "n_H < n_th" so that the march reads ONE
// value per cell, and -inf in the halo.  Also the per-block partial sums of the ionised fraction 1 - x_HI
// for automerge.
template <typename T>
__global__ void prep_fields_kernel(const T *__restrict__ nH, const T *__restrict__ xHI, double *__restrict__ a,
                                   int nx, int ny, int nz, double n_th, int use_flag, int periodic,
                                   double *__restrict__ partial) {
    __shared__ double sh[256];
    double acc = 0.0;
    // one padded row (fixed j, k) per block iteration, threads along x: no division per cell, coalesced rows
    const long long px = nx + 2, py = ny + 2, pz = nz + 2, nrow = py * pz;
    for (long long row = blockIdx.x; row < nrow; row += gridDim.x) {
        long long j = row % py - 1, k = row / py - 1;
        const bool row_inside = j >= 0 && j < ny && k >= 0 && k < nz;
        if (periodic) { j = (j + ny) % ny; k = (k + nz) % nz; }       // halo = image of the opposite side
        const long long src = (k * ny + j) * nx, dst = row * px;
        for (int ip = threadIdx.x; ip < (int)px; ip += blockDim.x) {
            int i = ip - 1;
            const bool inside = row_inside && i >= 0 && i < nx;
            double v = -CUDART_INF;
            if (periodic) i = i < 0 ? nx - 1 : (i >= nx ? 0 : i);
            if (inside || periodic) {
                const double n = (double)nH[src + i], x = (double)xHI[src + i];
                v = n * x;
                if (use_flag && !(n >= n_th)) v = -v;
                if (inside) acc += 1.0 - x;
            }
            a[dst + ip] = v;
        }
    }
    sh[threadIdx.x] = acc;
    __syncthreads();
    for (int o = blockDim.x >> 1; o > 0; o >>= 1) {
        if ((int)threadIdx.x < o) sh[threadIdx.x] += sh[threadIdx.x + o];
        __syncthreads();
    }
    if (threadIdx.x == 0) partial[blockIdx.x] = sh[0];
}

// fixed-order sum of the partials (deterministic)
__global__ void sum_partials_kernel(const double *partial, int n, double *out) {
    __shared__ double sh[256];
    double acc = 0.0;
    for (int i = threadIdx.x; i < n; i += blockDim.x) acc += partial[i];
    sh[threadIdx.x] = acc;
    __syncthreads();
    for (int o = blockDim.x >> 1; o > 0; o >>= 1) {
        if ((int)threadIdx.x < o) sh[threadIdx.x] += sh[threadIdx.x + o];
        __syncthreads();
    }
    if (threadIdx.x == 0) *out = sh[0];
}

// ---------------------------------------------------------------------------------------------------
// Finalise (row a9): Gamma = photons / (n_HI V) (Eq. 1 with V_box); heating (H1);
// per-block partial sums of the deposited photons for the budget.  Reads the padded accumulator and
// absorber, writes the caller's dense [nz][ny][nx] outputs.
__global__ void finalise_kernel(double *__restrict__ gamma, double *__restrict__ heat, const double *__restrict__ acc,
                                const double *__restrict__ absorber, int nx, int ny, int nz, double V,
                                double e_excess, int periodic, double *__restrict__ photons_out,
                                double *__restrict__ partial) {
    __shared__ double sh[256];
    double sum = 0.0;
    const long long px = nx + 2, pxy = (long long)(nx + 2) * (ny + 2), nrow = (long long)ny * nz;
    for (long long row = blockIdx.x; row < nrow; row += gridDim.x)
    for (int i = threadIdx.x; i < nx; i += blockDim.x) {             // one row (fixed j, k) per block iteration
        const long long j = row % ny, k = row / ny;
        const long long t = row * nx + i;
        const long long q = (k + 1) * pxy + (j + 1) * px + (i + 1);
        double ph = acc[q];
        if (periodic) {
            // neighbour shares deposited across a box face went to the halo image of the cell on the
            // opposite side: fold them back (only face halos can hold any: a neighbour differs in one axis)
            if (i == 0) ph += acc[q + nx];
            if (i == nx - 1) ph += acc[q - nx];
            if (j == 0) ph += acc[q + ny * px];
            if (j == ny - 1) ph += acc[q - ny * px];
            if (k == 0) ph += acc[q + nz * pxy];
            if (k == nz - 1) ph += acc[q - nz * pxy];
        }
        sum += ph;
        if (photons_out) { photons_out[t] = ph; continue; }     // shard mode: raw photon counts, reduced across GPUs first
        double g = 0.0, h = 0.0;
        if (ph != 0.0) {
            g = ph / (fabs(absorber[q]) * V);
            h = e_excess * ph / V;
        }
        gamma[t] = g;
        if (heat) heat[t] = h;
    }
    sh[threadIdx.x] = sum;
    __syncthreads();
    for (int o = blockDim.x >> 1; o > 0; o >>= 1) {
        if ((int)threadIdx.x < o) sh[threadIdx.x] += sh[threadIdx.x + o];
        __syncthreads();
    }
    if (threadIdx.x == 0) partial[blockIdx.x] = sh[0];
}

// Finalise from a dense [nz][ny][nx] photon grid (the all-reduced sum of the shards' grids)
__global__ void finalise_dense_kernel(double *__restrict__ gamma, double *__restrict__ heat,
                                      const double *__restrict__ photons, const double *__restrict__ absorber, int nx,
                                      int ny, int nz, double V, double e_excess, double *__restrict__ partial) {
    __shared__ double sh[256];
    double sum = 0.0;
    const long long px = nx + 2, pxy = (long long)(nx + 2) * (ny + 2), nrow = (long long)ny * nz;
    for (long long row = blockIdx.x; row < nrow; row += gridDim.x)
    for (int i = threadIdx.x; i < nx; i += blockDim.x) {             // one row (fixed j, k) per block iteration
        const long long j = row % ny, k = row / ny;
        const long long t = row * nx + i;
        const long long q = (k + 1) * pxy + (j + 1) * px + (i + 1);
        const double ph = photons[t];
        sum += ph;
        double g = 0.0, h = 0.0;
        if (ph != 0.0) {
            g = ph / (fabs(absorber[q]) * V);
            h = e_excess * ph / V;
        }
        gamma[t] = g;
        if (heat) heat[t] = h;
    }
    sh[threadIdx.x] = sum;
    __syncthreads();
    for (int o = blockDim.x >> 1; o > 0; o >>= 1) {
        if ((int)threadIdx.x < o) sh[threadIdx.x] += sh[threadIdx.x + o];
        __syncthreads();
    }
    if (threadIdx.x == 0) partial[blockIdx.x] = sh[0];
}

__global__ void pix2dir_kernel(int level, long long pix0, long long n, double *out) {
    const long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n) return;
    double x, y, z;
    pix2dir(level, (uint32_t)(pix0 + i), x, y, z);
    out[3 * i] = x; out[3 * i + 1] = y; out[3 * i + 2] = z;
}

}  // namespace nyxrt
