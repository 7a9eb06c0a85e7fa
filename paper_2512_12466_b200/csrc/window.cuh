// The march in windows of a shared geometry (open box, monochromatic): DESIGN.md rows a5-a7, third generation.
//
// Sources sit at cell centres and the geometry is source-relative (DESIGN.md DEC list, reading R13), so the GEOMETRY
// of a ray (level, pixel) -- the cells it crosses relative to its source, every ds, the nearest face, f_c, the
// distance at which it splits -- is bit for bit the same for every source.  Round 2's first attempts to use that
// marched the rays of several sources in lock step and lost to lane occupancy (a finished ray could not be replaced
// mid-way: profiles/r2_shared_geometry_experiment.md).  Here the sharing is in SPACE AND TIME at once:
//
//   - a batch is (stably) sorted by pixel GROUP (64 consecutive nested pixels: a compact patch of the sphere); a block
//     takes the rays of one group -- any number, from any sources -- and marches them WINDOW by window of 16 cells;
//   - per window, 64 threads run the geometry stage of march_kernel (3-D DDA, Eq. 5-8 geometry, Eq. 4 test: the
//     two thirds of the per-ray kernel's instructions) ONCE per pixel and leave 16 step descriptors per pixel in
//     shared memory; then every ray of the group that is still alive runs the physics stage (gather, dtau, exponential,
//     deposits) through those 16 steps, 128 rays per pass, its state parked in a block-private list between windows;
//   - all rays of a pass stand at the same window, so a lane that finishes a ray takes the next one of the list:
//     lanes idle for the rest of one 16-cell pass at most.
//
// Order of the tests per cell, the DEC arithmetic, the counters and the child slabs are those of march_kernel.
// Compiled with -fmad=false.
#pragma once
#include "march.cuh"

namespace nyxrt {

constexpr int WIN_THREADS = 128;
constexpr int WIN_WARPS = WIN_THREADS / 32;
constexpr int WIN_MIN_BLOCKS = 5;
constexpr int WIN_PIX = 64;               // pixels of a group
constexpr int WIN_PIX_BITS = 6;
constexpr int WIN_STEPS = 16;             // cells of a window
constexpr int WIN_CHUNK = 1024;           // entries of the sorted batch a block claims at a time
constexpr uint32_t WIN_NONE = 0xffffffffu;

// one cell of one pixel's ray as the geometry stage describes it
struct WinStep {
    double ds;            // segment length; 0: the cell is only touched at an edge / corner; -1: the cell's entry distance
                          // meets Eq. 4: the ray splits here instead of marching
    double fc;            // f_c = 1/2 + D_edge / L_pix of Eq. 5 / 7 (used when offn != off)
    int off, offn;        // the cell and the neighbour across the nearest face, as offsets from the source's cell
                          // (padded linear index); offn == off: D_edge >= L_pix / 2, no neighbour
};

// Sort keys of the batch the scheduler picked: key = pixel group, value = position in the batch; holes (slab padding)
// and the tail of the fixed-size buffer get keys above every group.
__global__ void window_keys_kernel(const LoopState *ls, RayPool pool, uint32_t *key_in, uint32_t *val_in, long long cap,
                                   uint32_t sentinel) {
    const long long batch = ls->batch, begin = ls->begin;
    for (long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x; i < cap; i += (long long)gridDim.x * blockDim.x) {
        uint32_t k = sentinel + 1u, v = WIN_NONE;
        if (i < batch) {
            const unsigned long long rk = pool.key[begin + i];
            k = rk == KEY_HOLE ? sentinel : (key_pix(rk) >> WIN_PIX_BITS);
            v = (uint32_t)i;
        }
        key_in[i] = k;
        val_in[i] = v;
    }
}

struct WinArgs {
    MarchArgs m;
    const uint32_t *gkey;                 // sorted group keys of the batch
    const uint32_t *order;                // their positions in the batch
    unsigned long long *lkey;             // block-private lists of the rays alive between two windows: [block][2][WIN_CHUNK]
    double *ltau, *lN;
    int *lbase;
    uint32_t hole_key;                    // the key holes were given
};

__global__ void __launch_bounds__(WIN_THREADS, WIN_MIN_BLOCKS) window_march_kernel(const __grid_constant__ WinArgs WA) {
    const MarchArgs &A = WA.m;
    // the window's step descriptors, one array per field (8-byte stride across pixels: no bank conflicts)
    __shared__ double Tds[WIN_STEPS][WIN_PIX], Tfc[WIN_STEPS][WIN_PIX];
    __shared__ int2 Toff[WIN_STEPS][WIN_PIX];                                     // x = off, y = offn
    __shared__ double gs[WIN_PIX], god[3][WIN_PIX], gsx[3][WIN_PIX], gd[3][WIN_PIX], ginv[3][WIN_PIX];
    __shared__ int goff[WIN_PIX], go[3][WIN_PIX], gstate[WIN_PIX];            // gstate: 0 no ray, 1 marching, 2 split reached
    __shared__ double Tesc[WIN_THREADS], Tres[WIN_THREADS];
    __shared__ WarpScratch W;
    __shared__ int s_end, s_next, s_any;
    __shared__ unsigned long long s_chunk;
    const LoopState *ls = A.ls;
    const long long batch = ls->batch;
    if (batch == 0) return;
    const int level = ls->level;
    const long long begin = ls->begin;
    const int tid = threadIdx.x, lane = tid & 31, wid = tid >> 5;
    const unsigned lt = (1u << lane) - 1u, FULL = 0xffffffffu;
    const double r2s = A.r2_split[level], Kl = A.K[level];
    const double Kh = 0.5 * A.K[level];
    const double tau_max = A.tau_max, sdx = A.sdx;
    const int sy = (int)A.px, sz = (int)A.pxy;
    const double *__restrict__ absorber = A.absorber;
    double *__restrict__ acc = A.acc;
    const bool lmax = level >= A.level_max;
    unsigned long long *lkey = WA.lkey + (size_t)blockIdx.x * 2 * WIN_CHUNK;
    double *ltau = WA.ltau + (size_t)blockIdx.x * 2 * WIN_CHUNK, *lN = WA.lN + (size_t)blockIdx.x * 2 * WIN_CHUNK;
    int *lbase = WA.lbase + (size_t)blockIdx.x * 2 * WIN_CHUNK;

    Tesc[tid] = 0.0;
    Tres[tid] = 0.0;
    unsigned int n_seg = 0, n_zero = 0, n_nbr = 0;
    if (lane == 0) {
        W.slab_pos[wid] = W.slab_end[wid] = 0;
        W.n_split[wid] = W.n_ktau[wid] = W.n_exit[wid] = W.n_klmax[wid] = W.n_hole[wid] = 0u;
    }
    __syncthreads();

    // retire the rays of a pass whose outcome is known (all lanes of the warp call it): march_kernel's retire
    auto retire = [&](int outcome, double rs, double rtau, double rN, unsigned long long rkey) {
        const unsigned m_any = __ballot_sync(FULL, outcome != OUT_NONE);
        if (m_any == 0) return;
        const unsigned m_split = __ballot_sync(FULL, outcome == OUT_SPLIT);
        const unsigned m_ktau = __ballot_sync(FULL, outcome == OUT_KILL_TAU);
        const unsigned m_exit = __ballot_sync(FULL, outcome == OUT_EXIT);
        const unsigned m_klmax = __ballot_sync(FULL, outcome == OUT_KILL_LMAX);
        if (lane == 0) {
            W.n_split[wid] += __popc(m_split); W.n_ktau[wid] += __popc(m_ktau); W.n_exit[wid] += __popc(m_exit);
            W.n_klmax[wid] += __popc(m_klmax);
        }
        if (outcome == OUT_EXIT) Tesc[tid] += rN;
        else if (outcome == OUT_KILL_TAU || outcome == OUT_KILL_LMAX) Tres[tid] += rN;
        if (m_split) {
            const int need = 4 * __popc(m_split);
            long long slab_pos = W.slab_pos[wid], slab_end = W.slab_end[wid];
            __syncwarp();
            const long long rem = slab_end - slab_pos;
            long long base = 0;
            if (need > rem) {
                if (lane == 0) base = (long long)atomicAdd((unsigned long long *)&A.ls->count[level + 1], (unsigned long long)CHILD_SLAB);
                base = __shfl_sync(FULL, base, 0);
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
                const double Nc = rN * 0.25;                                     // L shared evenly
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

    const long long nchunk = (batch + WIN_CHUNK - 1) / WIN_CHUNK;
    for (;;) {
        __syncthreads();
        if (tid == 0) s_chunk = atomicAdd((unsigned long long *)&A.ls->fetch, 1ull);
        __syncthreads();
        const long long ck = (long long)s_chunk;
        if (ck >= nchunk) break;
        const long long cbase = ck * WIN_CHUNK;
        const int n_chunk = (int)(batch - cbase < WIN_CHUNK ? batch - cbase : WIN_CHUNK);
        int a = 0;
        while (a < n_chunk) {
            // ---- the run of entries [a, b) with the same pixel group -----------------------------------------
            const uint32_t g = WA.gkey[cbase + a];
            if (tid == 0) { s_end = n_chunk; s_next = 0; }
            if (tid < WIN_PIX) gstate[tid] = 0;
            __syncthreads();
            for (int i = a + 1 + tid; i < n_chunk; i += WIN_THREADS)
                if (WA.gkey[cbase + i] != g) { atomicMin(&s_end, i); break; }
            __syncthreads();
            const int b = s_end;
            if (g >= WA.hole_key) {                                               // slab padding (sorted to the end): not rays
                if (g == WA.hole_key && tid == 0) W.n_hole[0] += (unsigned)(b - a);
                a = b;
                continue;
            }
            // pixels that have rays, and the distance at which their rays were born (the parent's split distance:
            // geometry, the same for every source)
            for (int i = a + tid; i < b; i += WIN_THREADS) {
                const long long slot = begin + (long long)WA.order[cbase + i];
                const int pl = (int)(key_pix(A.pool.key[slot]) & (WIN_PIX - 1));
                gs[pl] = A.pool.s[slot];
                gstate[pl] = 1;
            }
            __syncthreads();
            if (tid < WIN_PIX && gstate[tid] == 1) {
                double e0, e1, e2;
                pix2dir(level, (g << WIN_PIX_BITS) + (uint32_t)tid, e0, e1, e2);
                const double s = gs[tid];
                // O4: start-of-life cell, source-relative (source at its cell centre), rule R12
                double q, o0, o1, o2;
                q = fma(s, e0, 0.5); o0 = floor(q); if (q == o0 && e0 < 0.0) o0 -= 1.0;
                q = fma(s, e1, 0.5); o1 = floor(q); if (q == o1 && e1 < 0.0) o1 -= 1.0;
                q = fma(s, e2, 0.5); o2 = floor(q); if (q == o2 && e2 < 0.0) o2 -= 1.0;
                const double i0 = (e0 == 0.0) ? -CUDART_INF : 1.0 / e0;           // with od + (-0.5): s_x = +inf
                const double i1 = (e1 == 0.0) ? -CUDART_INF : 1.0 / e1;
                const double i2 = (e2 == 0.0) ? -CUDART_INF : 1.0 / e2;
                gd[0][tid] = e0; gd[1][tid] = e1; gd[2][tid] = e2;
                ginv[0][tid] = i0; ginv[1][tid] = i1; ginv[2][tid] = i2;
                god[0][tid] = o0; god[1][tid] = o1; god[2][tid] = o2;
                gsx[0][tid] = (o0 + signed_half(i0)) * i0;                       // ((o + [d > 0]) - 0.5) / d
                gsx[1][tid] = (o1 + signed_half(i1)) * i1;
                gsx[2][tid] = (o2 + signed_half(i2)) * i2;
                go[0][tid] = (int)o0; go[1][tid] = (int)o1; go[2][tid] = (int)o2;
                goff[tid] = (int)o2 * sz + (int)o1 * sy + (int)o0;
            }
            int n_cur = b - a, cur = 0;
            for (int win = 0;; ++win) {
                // ---- G stage: 16 cells of every pixel that still has rays (march_kernel's describe) -------------
                __syncthreads();
                if (tid < WIN_PIX && gstate[tid] == 1) {
                    double s = gs[tid], od0 = god[0][tid], od1 = god[1][tid], od2 = god[2][tid];
                    double sx0 = gsx[0][tid], sx1 = gsx[1][tid], sx2 = gsx[2][tid];
                    int off = goff[tid];
                    for (int j = 0; j < WIN_STEPS; ++j) {
                        WinStep D;
                        D.off = off; D.offn = off; D.fc = 1.0;
                        if (s * s > r2s) {                                        // Eq. 4 on the entry distance: the rays split here
                            // (the rest of the window repeats the cell: the look-ahead gathers stay on a valid address)
                            for (int jj = j; jj < WIN_STEPS; ++jj) { Tds[jj][tid] = -1.0; Tfc[jj][tid] = 1.0; Toff[jj][tid] = make_int2(off, off); }
                            gstate[tid] = 2;
                            break;
                        }
                        double s_exit = sx0; int ax = 0;
                        if (sx1 < s_exit) { s_exit = sx1; ax = 1; }
                        if (sx2 < s_exit) { s_exit = sx2; ax = 2; }               // first minimum, order x, y, z
                        double ds = s_exit - s;
                        if (!(ds > 0.0)) ds = 0.0;
                        D.ds = ds;
                        const double s_m = fma(0.5, ds, s);                       // = s + 0.5 ds (0.5 ds is exact)
                        double m0 = fma(s_m, gd[0][tid], 0.5) - od0;
                        double m1 = fma(s_m, gd[1][tid], 0.5) - od1;
                        double m2 = fma(s_m, gd[2][tid], 0.5) - od2;
                        // nearest face, first minimum in the order x-, x+, y-, y+, z-, z+
                        const double t0 = 1.0 - m0, t1 = 1.0 - m1, t2 = 1.0 - m2;
                        double h0 = m0; int f0 = -1;
                        if (t0 < h0) { h0 = t0; f0 = 1; }
                        double h1 = m1; int f1 = -sy;
                        if (t1 < h1) { h1 = t1; f1 = sy; }
                        double h2 = m2; int f2 = -sz;
                        if (t2 < h2) { h2 = t2; f2 = sz; }
                        double de = h0; int foff = f0;
                        if (h1 < de) { de = h1; foff = f1; }
                        if (h2 < de) { de = h2; foff = f2; }
                        if (de < 0.0) {
                            // rounding put the midpoint a hair outside the cell: redo with the clamp to [0, 1] of the DEC list
                            m0 = m0 < 0.0 ? 0.0 : (m0 > 1.0 ? 1.0 : m0);
                            m1 = m1 < 0.0 ? 0.0 : (m1 > 1.0 ? 1.0 : m1);
                            m2 = m2 < 0.0 ? 0.0 : (m2 > 1.0 ? 1.0 : m2);
                            de = m0; foff = -1;
                            double t = 1.0 - m0; if (t < de) { de = t; foff = 1; }
                            if (m1 < de) { de = m1; foff = -sy; }
                            t = 1.0 - m1; if (t < de) { de = t; foff = sy; }
                            if (m2 < de) { de = m2; foff = -sz; }
                            t = 1.0 - m2; if (t < de) { de = t; foff = sz; }
                        }
                        if (de < s_m * Kh && ds > 0.0) {                          // D_edge < L_pix / 2  (Eq. 5 / 7)
                            D.offn = off + foff;
                            D.fc = 0.5 + div_fast(de, s_m * Kl);                  // L_pix = s_m sqrt(Omega) (R22)
                        }
                        Tds[j][tid] = D.ds; Tfc[j][tid] = D.fc; Toff[j][tid] = make_int2(D.off, D.offn);
                        // advance one cell (DEC: s = s_exit; s_a = ((o_a + [d_a > 0]) - 0.5) / d_a)
                        s = s_exit;
                        const double iv = ginv[ax][tid];
                        const double one = signed_one(iv), half = signed_half(iv);
                        if (ax == 0) { od0 += one; sx0 = (od0 + half) * iv; }
                        if (ax == 1) { od1 += one; sx1 = (od1 + half) * iv; }
                        if (ax == 2) { od2 += one; sx2 = (od2 + half) * iv; }
                        const int ustp = ax == 0 ? 1 : (ax == 1 ? sy : sz);
                        off += __double2hiint(iv) < 0 ? -ustp : ustp;
                    }
                    gs[tid] = s; god[0][tid] = od0; god[1][tid] = od1; god[2][tid] = od2;
                    gsx[0][tid] = sx0; gsx[1][tid] = sx1; gsx[2][tid] = sx2;
                    goff[tid] = off;
                }
                if (tid == 0) s_next = 0;
                __syncthreads();
                // ---- P stage: every ray of the group that is still alive, 128 per pass --------------------------
                const int nxt = cur ^ 1;
                for (int i0 = 0; i0 < n_cur; i0 += WIN_THREADS) {
                    const int i = i0 + tid;
                    bool has = i < n_cur;
                    unsigned long long key = 0;
                    double tau = 0.0, N = 0.0;
                    int base = 0, pl = 0;
                    int outcome = OUT_NONE;
                    if (has) {
                        if (win == 0) {
                            const long long slot = begin + (long long)WA.order[cbase + a + i];
                            key = A.pool.key[slot];
                            tau = A.pool.tau[slot];
                            N = A.pool.N[slot];
                            pl = (int)(key_pix(key) & (WIN_PIX - 1));
                            const int4 sc = A.cat_cell[key_src(key)];
                            base = (sc.z + 1) * sz + (sc.y + 1) * sy + (sc.x + 1);
                            const int ci = sc.x + go[0][pl], cj = sc.y + go[1][pl], cq = sc.z + go[2][pl];
                            if (ci < 0 || ci >= A.nx || cj < 0 || cj >= A.ny || cq < 0 || cq >= A.nz) outcome = OUT_EXIT;   // born outside the box
                        } else {
                            key = lkey[cur * WIN_CHUNK + i];
                            tau = ltau[cur * WIN_CHUNK + i];
                            N = lN[cur * WIN_CHUNK + i];
                            base = lbase[cur * WIN_CHUNK + i];
                            pl = (int)(key_pix(key) & (WIN_PIX - 1));
                        }
                    }
                    if (has && outcome == OUT_NONE) {
                        // Gathers in bursts, one burst ahead: the cells of a window are known in advance (the window's
                        // table), so the absorbers -- cell and neighbour -- of four cells are requested back to back
                        // while the physics of the previous four runs.  Order matters: a warp has six scoreboards, and
                        // a wait for an old gather also waits for every newer one that shares its scoreboard; so a
                        // burst is first consumed (opacity per unit length, exit and neighbour flags), THEN the next
                        // burst is issued, then the physics runs on values that need no wait.  A ray that leaves the box
                        // may read, never use, up to seven cells beyond the halo: the guard band covers them.
                        constexpr int Q = 4;
                        double rc[Q], rn[Q];
#pragma unroll
                        for (int k = 0; k < Q; ++k) {
                            const int2 o = Toff[k][pl];
                            rc[k] = __ldg(absorber + (base + o.x));
                            rn[k] = o.y != o.x ? __ldg(absorber + (base + o.y)) : 0.0;
                        }
#pragma unroll
                        for (int q0 = 0; q0 < WIN_STEPS; q0 += Q) {
                            double a1[Q];
                            unsigned exm = 0, nbm = 0;
#pragma unroll
                            for (int k = 0; k < Q; ++k) {
                                a1[k] = fabs(rc[k]) * sdx;
                                exm |= (__double2hiint(rc[k]) == (int)0xfff00000 ? 1u : 0u) << k;     // the halo holds -inf
                                nbm |= (rn[k] > 0.0 ? 1u : 0u) << k;              // in the box, absorber > 0, n_H >= n_th
                            }
                            asm volatile("" ::: "memory");
                            if (q0 + Q < WIN_STEPS) {
#pragma unroll
                                for (int k = 0; k < Q; ++k) {
                                    const int2 o = Toff[q0 + Q + k][pl];
                                    rc[k] = __ldg(absorber + (base + o.x));
                                    rn[k] = o.y != o.x ? __ldg(absorber + (base + o.y)) : 0.0;
                                }
                            }
                            asm volatile("" ::: "memory");
#pragma unroll
                            for (int k = 0; k < Q; ++k) {
                                const int j = q0 + k;
                                const int2 o = Toff[j][pl];
                                const double ds = Tds[j][pl];
                                outcome = ((exm >> k) & 1u) ? OUT_EXIT : (tau >= tau_max ? OUT_KILL_TAU : (lmax ? OUT_KILL_LMAX : (ds < 0.0 ? OUT_SPLIT : OUT_NONE)));
                                if (outcome != OUT_NONE) break;
                                if (ds > 0.0) {
                                    ++n_seg;
                                    const double dtau = a1[k] * ds;
                                    double pm, left;
                                    absorb_fraction(dtau, pm, left);
                                    const double dN = N * (-pm);
                                    if (dN > 0.0) {
                                        double fc = 1.0;
                                        if (o.y != o.x && ((nbm >> k) & 1u)) {
                                            fc = Tfc[j][pl];
                                            ++n_nbr;
                                            atomicAdd(acc + (base + o.y), (1.0 - fc) * dN);
                                        }
                                        atomicAdd(acc + (base + o.x), fc * dN);
                                    }
                                    N = N * left;
                                    tau = tau + dtau;
                                } else {
                                    ++n_zero;
                                }
                            }
                            if (outcome != OUT_NONE) break;
                        }
                    }
                    // survivors wait for the next window in the block's list
                    const bool live = has && outcome == OUT_NONE;
                    const unsigned m_live = __ballot_sync(FULL, live);
                    int pos = 0;
                    if (lane == 0 && m_live) pos = atomicAdd(&s_next, __popc(m_live));
                    pos = __shfl_sync(FULL, pos, 0);
                    if (live) {
                        const int q = nxt * WIN_CHUNK + pos + __popc(m_live & lt);
                        lkey[q] = key; ltau[q] = tau; lN[q] = N; lbase[q] = base;
                    }
                    retire(has ? outcome : OUT_NONE, gs[pl], tau, N, key);
                }
                __syncthreads();
                n_cur = s_next;
                cur = nxt;
                if (n_cur == 0) break;
            }
            a = b;
        }
    }
    // pad the unused tail of the last child slab
    __syncwarp();
    for (long long h = W.slab_pos[wid] + lane; h < W.slab_end[wid]; h += 32) A.pool.key[A.pool.off[level + 1] + h] = KEY_HOLE;

    unsigned long long seg64 = n_seg, zero64 = n_zero, nbr64 = n_nbr;
    double esc = Tesc[tid], res = Tres[tid];
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) {
        seg64 += __shfl_xor_sync(FULL, seg64, o);
        zero64 += __shfl_xor_sync(FULL, zero64, o);
        nbr64 += __shfl_xor_sync(FULL, nbr64, o);
        esc += __shfl_xor_sync(FULL, esc, o);
        res += __shfl_xor_sync(FULL, res, o);
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
    }
}

}  // namespace nyxrt
