// The ray loop on shared geometry (open box): march + deposit + filter + split of DESIGN.md rows a4-a8, second
// generation.
//
// Why.  Sources sit at cell centres and the geometry is written in source-relative coordinates (DESIGN.md DEC
// list, reading R13), so everything that is GEOMETRY of a ray (level, pixel) -- the cells it crosses relative to
// its source, every segment length ds, the nearest face, f_c of Eq. 5 / 7, the distance at which it splits
// (Eq. 4) -- is bit for bit the same for EVERY source.  Only the absorber values along the way, tau, the photon
// count and "did it leave the box / run out of photons" belong to a single ray.
//
// The ray store holds QUADS: the four children of one split share the source, the distance
// travelled, the optical depth and the photon share at birth, so they are one 32-byte record keyed by the
// parent's pixel.  A batch of quads is sorted by that key; quads of different sources with the same key then sit
// side by side.  A warp is 8 columns of 4 lanes: a column takes up to RMAX quads with the same key, lane j of
// the column marches child pixel 4 key + j for all of them in lock step: per cell the geometry stage (3-D DDA,
// Eq. 5-8 geometry, Eq. 4 test: ~130 instructions, two thirds of the per-ray kernel) runs ONCE per lane and the
// physics stage (gather, dtau, exponential, deposits: ~60 instructions) once per ray.  The rays of one lane also
// give the fp64 pipe independent dependency chains.  Survivors are repacked at every level (the sort), so the
// lanes of a column start full whatever happened to the rays' ancestors.
//
// Deposits along a ray are combined before they reach memory: the neighbour c' of Eq. 6 / 8 is, for 81 % of
// the neighbour deposits (measured on levels 7 and 9), the cell the ray has just left or the one it enters
// next, so a cell's RED is held back one step and collects its own share f_c dN plus the (1 - f_c) dN shares
// of the steps before and after: 1.14 RED per segment instead of 1.75, and the absorber of c' is then a value
// the ray loads anyway (1.14 gathers per segment instead of 1.75).  Only the summation order changes.
//
// Order of the tests per cell, the DEC arithmetic and the counters are those of march.cuh / the oracle
// (box exit, tau >= tau_max, l_max, split, segment).  Compiled with -fmad=false.
#pragma once
#include "march.cuh"

namespace nyxrt {

constexpr int BUNDLE_THREADS = 128;
constexpr int BUNDLE_WARPS = BUNDLE_THREADS / 32;
constexpr int BUNDLE_MIN_BLOCKS = 3;
constexpr int BUNDLE_RMAX = 4;            // rays of different sources that one lane marches together
constexpr uint32_t ORDER_NONE = 0xffffffffu;

// ---------------------------------------------------------------------------------------------------
// Emit (PAPER.md:111, 203 spawn_rays): three level-0 quads per catalogue source = the 12 level-0 pixels, L/12
// each.  Source sharding as in emit_kernel.
__global__ void bundle_emit_kernel(const LoopState *ls, QuadPool qp, const double *cat_L, int rank, int world) {
    const long long n = 3 * ls->emit_n;
    const long long src0 = ls->emit_src, slot0 = ls->emit_slot;
    for (long long r = (long long)blockIdx.x * blockDim.x + threadIdx.x; r < n; r += (long long)gridDim.x * blockDim.x) {
        const long long a = (src0 + r / 3) * world + rank;
        const long long t = slot0 + r;
        qp.key[t] = (uint32_t)(r % 3);
        qp.src[t] = (uint32_t)a;
        qp.s[t] = 0.0;
        qp.tau[t] = 0.0;
        qp.N[t] = cat_L[a] / 12.0;
    }
}

// Sort keys of the batch the scheduler picked: (parent pixel, rank of the source along a Morton curve through the
// box), value = position in the batch; the tail of the fixed-size sort buffer is filled with a key larger than any
// pixel.  Quads with the same pixel then sit side by side with their sources in spatial order: the rays one lane
// marches together start from neighbouring sources, meet the same structures and end at about the same step.
__global__ void bundle_keys_kernel(const LoopState *ls, QuadPool qp, long long cap, int rank_bits, uint64_t sentinel) {
    const long long batch = ls->batch, begin = ls->begin;
    for (long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x; i < cap; i += (long long)gridDim.x * blockDim.x) {
        const bool in = i < batch;
        qp.key_in[i] = in ? (((uint64_t)qp.key[begin + i] << rank_bits) | qp.src_rank[qp.src[begin + i]]) : sentinel;
        qp.val_in[i] = in ? (uint32_t)i : ORDER_NONE;
    }
}

// Morton key of a source's cell at a resolution of 2^shift cells (10 bits per axis) and the scatter of the sorted
// order into ranks.
__device__ __forceinline__ uint32_t spread3(uint32_t v) {
    v &= 0x3ffu;
    v = (v | (v << 16)) & 0x030000ffu;
    v = (v | (v << 8)) & 0x0300f00fu;
    v = (v | (v << 4)) & 0x030c30c3u;
    v = (v | (v << 2)) & 0x09249249u;
    return v;
}
__global__ void morton_kernel(const int4 *__restrict__ cell, long long n, int shift, int *__restrict__ key, int *__restrict__ idx) {
    const long long a = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (a >= n) return;
    const int4 c = cell[a];
    key[a] = (int)(spread3((uint32_t)c.x >> shift) | (spread3((uint32_t)c.y >> shift) << 1) | (spread3((uint32_t)c.z >> shift) << 2));
    idx[a] = (int)a;
}
__global__ void rank_kernel(const int *__restrict__ sorted_idx, long long n, uint32_t *__restrict__ rank) {
    const long long a = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (a < n) rank[sorted_idx[a]] = (uint32_t)a;
}

// One ray-cell step as the geometry stage describes it; shared by the rays of all bundles in a lane.
template <typename IDX>
struct StepDesc {
    double ds;            // segment length (0: the cell is only touched at an edge / corner)
    double fc, omf;       // f_c = 1/2 + D_edge / L_pix (Eq. 5 / 7) and 1 - f_c, valid when nbk != 0
    IDX off;              // the cell, as an offset from the source's cell (padded linear index)
    IDX offp;             // the cell of the previous step
    IDX offn;             // the neighbour across the nearest face
    int flag;             // 1: the entry distance meets Eq. 4: the ray splits here instead of marching
    int nbk;              // neighbour: 0 none (D_edge >= L_pix / 2), 1 the next cell of the ray, 2 the previous one, 3 another
};

// GEOM: 0 no correction, 1 Eq. 5 only, 3 Eq. 5-6 / 7-8, 4 squared (as march_kernel).  LUT: spectrum table.
template <int GEOM, typename IDX, bool LUT, int RMAX>
__global__ void __launch_bounds__(BUNDLE_THREADS, BUNDLE_MIN_BLOCKS) bundle_march_kernel(const __grid_constant__ MarchArgs A) {
    __shared__ double Td[3][BUNDLE_THREADS], Tinv[3][BUNDLE_THREADS];     // the lane's direction and 1/d
    __shared__ double Tesc[BUNDLE_THREADS], Tres[BUNDLE_THREADS];
    const LoopState *ls = A.ls;
    const long long batch = ls->batch;
    if (batch == 0) return;
    const int level = ls->level;
    const long long begin = ls->begin;
    const int lane = threadIdx.x & 31;
    const unsigned lt = (1u << lane) - 1u;
    const double r2s = A.r2_split[level], Kl = A.K[level];
    const double Kh = 0.5 * A.K[level];
    const double tau_max = A.tau_max, sdx = A.sdx;
    const IDX sy = (IDX)A.px, sz = (IDX)A.pxy;
    const double *__restrict__ absorber = A.absorber;
    double *__restrict__ acc = A.acc;
    const QuadPool &qp = A.qp;
    const bool lmax = level >= A.level_max;
    const unsigned FULL = 0xffffffffu;

    Tesc[threadIdx.x] = 0.0;
    Tres[threadIdx.x] = 0.0;
    unsigned int n_seg = 0, n_zero = 0, n_nbr = 0;
    double lost = 0.0;
    unsigned int w_spawn = 0, w_split = 0, w_ktau = 0, w_exit = 0, w_klmax = 0;    // warp-uniform tallies

#ifdef NYXRT_DIAG
    unsigned long long dg_rounds = 0, dg_tasks = 0, dg_quads = 0, dg_steps = 0, dg_slotsteps = 0, dg_lanesteps = 0;
#endif
    const long long nwin = (batch + 31) / 32;
    for (;;) {
        unsigned long long w = 0;
        if (lane == 0) w = atomicAdd((unsigned long long *)&A.ls->fetch, 1ull);
        w = __shfl_sync(FULL, w, 0);
        if ((long long)w >= nwin) break;
        // the window: 32 consecutive quads of the (sorted) batch, one per lane.  A TASK is a run of up to RMAX
        // quads with the same key (= quads of different sources, the same four pixels); a column (4 lanes)
        // marches one task per round.
        uint32_t ent = ORDER_NONE, ent_key = 0;
        if ((long long)w * 32 + lane < batch) {
            ent = A.order ? A.order[w * 32 + lane] : (uint32_t)(w * 32 + lane);
            if (ent != ORDER_NONE) ent_key = qp.key[begin + ent];
        }
        const unsigned valid = __ballot_sync(FULL, ent != ORDER_NONE);
        const uint32_t key_left = __shfl_up_sync(FULL, ent_key, 1);
        const unsigned heads = __ballot_sync(FULL, lane == 0 || ent_key != key_left) | 1u;
        const int run0 = 31 - __clz(heads & ((lt << 1) | 1u));               // first lane of this lane's run
        const unsigned tasks = __ballot_sync(FULL, ent != ORDER_NONE && ((lane - run0) % RMAX) == 0);
        const int ntask = __popc(tasks), nvalid = __popc(valid);
        w_spawn += 4u * (unsigned)nvalid;
#ifdef NYXRT_DIAG
        dg_tasks += ntask; dg_quads += nvalid;
#endif
        for (int round = 0; 8 * round < ntask; ++round) {
            // ---- column set-up: up to RMAX quads of different sources, the same four pixels ------------------
            const int t = 8 * round + (lane >> 2);
            int first = 0, len = 0;
            if (t < ntask) {
                first = __fns(tasks, 0, t + 1);
                len = (t + 1 < ntask ? (int)__fns(tasks, 0, t + 2) : nvalid) - first;
            }
            const uint32_t pix = 4u * __shfl_sync(FULL, ent_key, first) + (uint32_t)(lane & 3);
            uint32_t src[RMAX];
            IDX base[RMAX];
            double tau[RMAX], N[RMAX], pend[RMAX], carry[RMAX], a0[RMAX], a1[RMAX], wsh[RMAX];
            unsigned alive = 0;                      // bit r: this lane's ray of quad r is marching
            unsigned pe = 0;                         // bit r: the previous cell can take a neighbour share
            unsigned o_split = 0, o_ktau = 0, o_exit = 0, o_klmax = 0;     // bit r: how the ray ended
            double s = 0.0;
            int4 sc[RMAX];
#pragma unroll
            for (int r = 0; r < RMAX; ++r) {
                src[r] = 0; base[r] = 0; tau[r] = 0.0; N[r] = 0.0; pend[r] = 0.0; carry[r] = 0.0; a0[r] = 0.0; a1[r] = 0.0;
                wsh[r] = 0.0;
                sc[r] = make_int4(0, 0, 0, 0);
                const uint32_t e = __shfl_sync(FULL, ent, (first + r) & 31);
                if (r < len) {
                    const long long q = begin + (long long)e;
                    src[r] = qp.src[q];
                    s = qp.s[q];
                    tau[r] = qp.tau[q];
                    N[r] = qp.N[q];
                    sc[r] = A.cat_cell[src[r]];
                    alive |= 1u << r;
                }
            }
            const int R = __reduce_max_sync(FULL, len);   // slots in use in this round (warp-uniform)
            double od0, od1, od2, sx0, sx1, sx2;
            IDX off, offp, pstp = 0;
            {
                double e0 = 0.0, e1 = 0.0, e2 = 0.0;
                if (alive) pix2dir(level, pix, e0, e1, e2);
                // O4: start-of-life cell, source-relative (source at its cell centre), rule R12
                double q;
                q = fma(s, e0, 0.5); od0 = floor(q); if (q == od0 && e0 < 0.0) od0 -= 1.0;
                q = fma(s, e1, 0.5); od1 = floor(q); if (q == od1 && e1 < 0.0) od1 -= 1.0;
                q = fma(s, e2, 0.5); od2 = floor(q); if (q == od2 && e2 < 0.0) od2 -= 1.0;
                const double i0 = (e0 == 0.0) ? -CUDART_INF : 1.0 / e0;           // with od + (-0.5): s_x = +inf
                const double i1 = (e1 == 0.0) ? -CUDART_INF : 1.0 / e1;
                const double i2 = (e2 == 0.0) ? -CUDART_INF : 1.0 / e2;
                Td[0][threadIdx.x] = e0; Td[1][threadIdx.x] = e1; Td[2][threadIdx.x] = e2;
                Tinv[0][threadIdx.x] = i0; Tinv[1][threadIdx.x] = i1; Tinv[2][threadIdx.x] = i2;
                sx0 = (od0 + signed_half(i0)) * i0;                              // ((o + [d > 0]) - 0.5) / d
                sx1 = (od1 + signed_half(i1)) * i1;
                sx2 = (od2 + signed_half(i2)) * i2;
                const long long o0 = (long long)od0, o1 = (long long)od1, o2 = (long long)od2;
                off = (IDX)(o2 * (long long)sz + o1 * (long long)sy + o0);
                offp = off;
#pragma unroll
                for (int r = 0; r < RMAX; ++r) {
                    base[r] = (IDX)(((long long)sc[r].z + 1) * (long long)sz + ((long long)sc[r].y + 1) * (long long)sy + sc[r].x + 1);
                    if (LUT && ((alive >> r) & 1u)) { wsh[r] = N[r]; N[r] = lut_q(A, tau[r]); }
                    const long long ci = sc[r].x + o0, cj = sc[r].y + o1, ck = sc[r].z + o2;
                    if (((alive >> r) & 1u) && (ci < 0 || ci >= A.nx || cj < 0 || cj >= A.ny || ck < 0 || ck >= A.nz)) {
                        // born outside the box: leaves at once with no segment (oracle: the test before the loop)
                        Tesc[threadIdx.x] += LUT ? wsh[r] * (1.0 - N[r]) : N[r];
                        o_exit |= 1u << r;
                        alive &= ~(1u << r);
                    }
                }
            }

            // G stage: describe the cell the DDA stands in (geometry only), advance the DDA.  A cell whose entry
            // distance meets Eq. 4 is only flagged: the DDA stays put, so that the children inherit s.
            auto describe = [&](StepDesc<IDX> &D) {
                D.off = off;
                D.offp = offp;
                D.offn = off;
                D.flag = s * s > r2s ? 1 : 0;
                D.nbk = 0;
                D.ds = 0.0;
                D.fc = 1.0;
                D.omf = 0.0;
                if (D.flag) return;
                double s_exit = sx0; int ax = 0;
                if (sx1 < s_exit) { s_exit = sx1; ax = 1; }
                if (sx2 < s_exit) { s_exit = sx2; ax = 2; }                       // first minimum, order x, y, z
                double ds = s_exit - s;
                if (!(ds > 0.0)) ds = 0.0;
                D.ds = ds;
                const double iv = Tinv[ax][threadIdx.x];
                const IDX ustp = ax == 0 ? (IDX)1 : (ax == 1 ? sy : sz);
                const IDX stp = __double2hiint(iv) < 0 ? -ustp : ustp;          // 1/d < 0: the ray moves down the axis
                if (GEOM != 0) {
                    const double s_m = fma(0.5, ds, s);                           // = s + 0.5 ds (0.5 ds is exact)
                    double m0 = fma(s_m, Td[0][threadIdx.x], 0.5) - od0;
                    double m1 = fma(s_m, Td[1][threadIdx.x], 0.5) - od1;
                    double m2 = fma(s_m, Td[2][threadIdx.x], 0.5) - od2;
                    // nearest face, first minimum in the order x-, x+, y-, y+, z-, z+
                    const double t0 = 1.0 - m0, t1 = 1.0 - m1, t2 = 1.0 - m2;
                    double h0 = m0; IDX f0 = (IDX)-1;
                    if (t0 < h0) { h0 = t0; f0 = (IDX)1; }
                    double h1 = m1; IDX f1 = -sy;
                    if (t1 < h1) { h1 = t1; f1 = sy; }
                    double h2 = m2; IDX f2 = -sz;
                    if (t2 < h2) { h2 = t2; f2 = sz; }
                    double de = h0; IDX foff = f0;
                    if (h1 < de) { de = h1; foff = f1; }
                    if (h2 < de) { de = h2; foff = f2; }
                    if (de < 0.0) {
                        // rounding put the midpoint a hair outside the cell: redo with the clamp to [0, 1] of the DEC list
                        m0 = m0 < 0.0 ? 0.0 : (m0 > 1.0 ? 1.0 : m0);
                        m1 = m1 < 0.0 ? 0.0 : (m1 > 1.0 ? 1.0 : m1);
                        m2 = m2 < 0.0 ? 0.0 : (m2 > 1.0 ? 1.0 : m2);
                        de = m0; foff = (IDX)-1;
                        double t = 1.0 - m0; if (t < de) { de = t; foff = (IDX)1; }
                        if (m1 < de) { de = m1; foff = -sy; }
                        t = 1.0 - m1; if (t < de) { de = t; foff = sy; }
                        if (m2 < de) { de = m2; foff = -sz; }
                        t = 1.0 - m2; if (t < de) { de = t; foff = sz; }
                    }
                    if (de < s_m * Kh && ds > 0.0) {                              // D_edge < L_pix / 2  (Eq. 5 / 7)
                        D.offn = off + foff;
                        D.nbk = foff == stp ? 1 : (foff == -pstp ? 2 : 3);        // pstp = 0 before the first step
                        D.fc = 0.5 + div_fast(de, s_m * Kl);                      // L_pix = s_m sqrt(Omega) (R22)
                        D.omf = 1.0 - D.fc;
                    }
                }
                // advance one cell (DEC: s = s_exit; s_a = ((o_a + [d_a > 0]) - 0.5) / d_a)
                s = s_exit;
                const double one = signed_one(iv), half = signed_half(iv);
                if (ax == 0) { od0 += one; sx0 = (od0 + half) * iv; }
                if (ax == 1) { od1 += one; sx1 = (od1 + half) * iv; }
                if (ax == 2) { od2 += one; sx2 = (od2 + half) * iv; }
                offp = off;
                off += stp;
                pstp = stp;
            };

            // gathers of one step: the cell's absorber for every marching ray
            auto gather = [&](const StepDesc<IDX> &D, double (&a)[RMAX]) {
#pragma unroll
                for (int r = 0; r < RMAX; ++r)
                    if ((alive >> r) & 1u) a[r] = __ldg(absorber + (base[r] + D.off));
            };

            // P stage for the rays of this lane at the step D: ac = absorbers of the cell, an = of the NEXT cell
            auto physics = [&](const StepDesc<IDX> &D, const double (&ac)[RMAX], const double (&an)[RMAX]) {
#pragma unroll
                for (int r = 0; r < RMAX; ++r) {
                    if (r >= R) break;                                             // warp-uniform
                    if (!((alive >> r) & 1u)) continue;
                    const double a_c = ac[r];
                    const bool f_exit = __double2hiint(a_c) == (int)0xfff00000;   // the halo holds -inf
                    if (!f_exit && !(tau[r] >= tau_max) && !lmax && !D.flag) {
                        double own = 0.0, S = 0.0;
                        if (D.ds > 0.0) {
                            ++n_seg;
                            const double dtau = (fabs(a_c) * sdx) * D.ds;
                            double pm, left, dN;
                            if constexpr (LUT) {
                                left = lut_q(A, tau[r] + dtau);                   // Q at the end of the segment
                                dN = wsh[r] * (left - N[r]);
                            } else {
                                absorb_fraction(dtau, pm, left);
                                dN = N[r] * (-pm);
                            }
                            if (dN > 0.0) {
                                own = dN;
                                if (GEOM == 3) {
                                    if (D.nbk != 0) {
                                        bool elig;                                 // in the box, absorber > 0, n_H >= n_th
                                        if (D.nbk == 1) elig = an[r] > 0.0;
                                        else if (D.nbk == 2) elig = (pe >> r) & 1u;
                                        else elig = __ldg(absorber + (base[r] + D.offn)) > 0.0;
                                        if (elig) { S = D.omf * dN; own = D.fc * dN; ++n_nbr; }
                                    }
                                } else if (GEOM == 1 || GEOM == 4) {
                                    if (D.nbk != 0) {
                                        const double fc = GEOM == 4 ? D.fc * D.fc : D.fc;
                                        own = fc * dN;
                                        lost += (1.0 - fc) * dN;
                                    }
                                }
                            }
                            N[r] = LUT ? left : N[r] * left;
                            tau[r] = tau[r] + dtau;
                        } else {
                            ++n_zero;
                        }
                        // the previous cell's total is complete now: its own share, what the step before it sent
                        // forward, and this step's share if its neighbour is the previous cell
                        const double v = D.nbk == 2 ? pend[r] + S : pend[r];
                        if (v != 0.0) atomicAdd(acc + (base[r] + D.offp), v);
                        pend[r] = own + carry[r];
                        carry[r] = D.nbk == 1 ? S : 0.0;
                        if (D.nbk == 3 && S != 0.0) atomicAdd(acc + (base[r] + D.offn), S);
                        pe = a_c > 0.0 ? (pe | (1u << r)) : (pe & ~(1u << r));
                    } else {
                        // the ray ends on entering this cell: what it still owes goes out, then the tallies
                        if (pend[r] != 0.0) atomicAdd(acc + (base[r] + D.offp), pend[r]);
                        if (carry[r] != 0.0) atomicAdd(acc + (base[r] + D.off), carry[r]);
                        const double rest = LUT ? wsh[r] * (1.0 - N[r]) : N[r];
                        if (f_exit) { o_exit |= 1u << r; Tesc[threadIdx.x] += rest; }
                        else if (tau[r] >= tau_max) { o_ktau |= 1u << r; Tres[threadIdx.x] += rest; }
                        else if (lmax) { o_klmax |= 1u << r; Tres[threadIdx.x] += rest; }
                        else o_split |= 1u << r;
                        alive &= ~(1u << r);
                    }
                }
            };

            // ---- march in lock step: the geometry runs one cell ahead of the physics ------------------------
            StepDesc<IDX> DA, DB;
            DB.ds = 0.0; DB.fc = 1.0; DB.omf = 0.0; DB.off = off; DB.offp = off; DB.offn = off; DB.flag = 0; DB.nbk = 0;
            describe(DA);
            gather(DA, a0);
#ifdef NYXRT_DIAG
            ++dg_rounds;
#endif
            while (__any_sync(FULL, alive != 0u)) {
#ifdef NYXRT_DIAG
                dg_steps += 2; dg_slotsteps += 2 * R; dg_lanesteps += __popc(__ballot_sync(FULL, alive != 0u));
#endif
                if (alive && !DA.flag) { describe(DB); gather(DB, a1); }
                physics(DA, a0, a1);
                if (alive && !DB.flag) { describe(DA); gather(DA, a0); }
                physics(DB, a1, a0);
            }

            // ---- tallies and the children of the rays that split: one quad per split ------------
            int n_child = 0;
            unsigned m_split[RMAX];
#pragma unroll
            for (int r = 0; r < RMAX; ++r) {
                m_split[r] = __ballot_sync(FULL, (o_split >> r) & 1u);
                n_child += __popc(m_split[r]);
                w_ktau += __popc(__ballot_sync(FULL, (o_ktau >> r) & 1u));
                w_exit += __popc(__ballot_sync(FULL, (o_exit >> r) & 1u));
                w_klmax += __popc(__ballot_sync(FULL, (o_klmax >> r) & 1u));
            }
            w_split += (unsigned)n_child;
            if (n_child) {
                long long cbase = 0;
                if (lane == 0) cbase = (long long)atomicAdd((unsigned long long *)&A.ls->count[level + 1], (unsigned long long)n_child);
                cbase = __shfl_sync(FULL, cbase, 0);
                if (cbase + n_child > qp.cap[level + 1]) {
                    if (lane == 0) A.ls->overflow = 1;
                } else {
                    long long ct = qp.off[level + 1] + cbase;
#pragma unroll
                    for (int r = 0; r < RMAX; ++r) {
                        if ((o_split >> r) & 1u) {
                            const long long q = ct + __popc(m_split[r] & lt);
                            qp.key[q] = pix;                                       // children: pixels 4 pix .. 4 pix + 3
                            qp.src[q] = src[r];
                            qp.s[q] = s;
                            qp.tau[q] = tau[r];
                            qp.N[q] = (LUT ? wsh[r] : N[r]) * 0.25;               // L shared evenly
                        }
                        ct += __popc(m_split[r]);
                    }
                }
            }
        }
    }

    // flush per-thread / per-warp tallies
    unsigned long long seg64 = n_seg, zero64 = n_zero, nbr64 = n_nbr;
    double esc = Tesc[threadIdx.x], res = Tres[threadIdx.x];
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) {
        seg64 += __shfl_xor_sync(FULL, seg64, o);
        zero64 += __shfl_xor_sync(FULL, zero64, o);
        nbr64 += __shfl_xor_sync(FULL, nbr64, o);
        esc += __shfl_xor_sync(FULL, esc, o);
        res += __shfl_xor_sync(FULL, res, o);
        lost += __shfl_xor_sync(FULL, lost, o);
    }
    if (lane == 0) {
        DevStats *ds = A.ds;
#ifdef NYXRT_DIAG
        atomicAdd(&ds->dg_rounds, dg_rounds); atomicAdd(&ds->dg_tasks, dg_tasks); atomicAdd(&ds->dg_quads, dg_quads);
        atomicAdd(&ds->dg_steps, dg_steps); atomicAdd(&ds->dg_slotsteps, dg_slotsteps); atomicAdd(&ds->dg_lanesteps, dg_lanesteps);
#endif
        if (seg64) atomicAdd(&ds->segments, seg64);
        if (zero64) atomicAdd(&ds->zero_len, zero64);
        if (nbr64) atomicAdd(&ds->nbr_deposits, nbr64);
        if (w_spawn) atomicAdd(&ds->spawned[level], (unsigned long long)w_spawn);
        if (w_split) atomicAdd(&ds->split[level], (unsigned long long)w_split);
        if (w_ktau) atomicAdd(&ds->killed_tau[level], (unsigned long long)w_ktau);
        if (w_exit) atomicAdd(&ds->exited[level], (unsigned long long)w_exit);
        if (w_klmax) atomicAdd(&ds->killed_lmax[level], (unsigned long long)w_klmax);
        if (esc != 0.0) atomicAdd(&ds->escaped, esc);
        if (res != 0.0) atomicAdd(&ds->residual, res);
        if (lost != 0.0) atomicAdd(&ds->lost, lost);
    }
}

}  // namespace nyxrt
