// The ray loop on the device: scheduler, emit, march+deposit+filter+split (SURVEY/DESIGN rows a4-a8).
//
// One launch marches a batch of rays that all sit on the SAME HEALPix level (the pool is one stack per
// level), so the split radius, the pixel width and the expected number of cells per ray are uniform
// across a launch.  Each ray is marched to its end: tau >= tau_max (filter), box exit
// (BASELINE.json configs; reading R20) or the split criterion Eq. 4, in which case the
// four children are pushed on the stack of level+1.
//
// Everything that steers control flow follows DESIGN.md's DEC list literally; this translation unit is
// compiled with -fmad=false.
#pragma once
#include "healpix.cuh"
#include "state.cuh"

namespace nyxrt {

constexpr int MARCH_THREADS = 256;

// ---------------------------------------------------------------------------------------------------
// Scheduler: one thread decides what the next emit + march launches do.
//   1. deepest level holding a full batch; else
//   2. if sources remain, top level 0 up with 12 rays per source, then 1. again; else
//   3. the shallowest non-empty level (drain).
// With caps of 2B (level 0) and 5B (deeper levels) no stack can overflow.
__global__ void sched_kernel(LoopState *ls, DevStats *ds, RayPool pool, int nlev) {
    if (threadIdx.x != 0 || blockIdx.x != 0) return;
    ls->emit_n = 0;
    ls->batch = 0;
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
    ls->iterations += 1;
    ds->spawned[pick] += (unsigned long long)b;          // every ray is marched exactly once
}

// ---------------------------------------------------------------------------------------------------
// Emit (PAPER.md:111, 203 spawn_rays): 12 level-0 rays per catalogue source, L/12 each.
__global__ void emit_kernel(const LoopState *ls, RayPool pool, const double *cat_L) {
    const long long n = ls->emit_n * 12;
    const long long src0 = ls->emit_src, slot0 = ls->emit_slot;
    for (long long r = (long long)blockIdx.x * blockDim.x + threadIdx.x; r < n;
         r += (long long)gridDim.x * blockDim.x) {
        const long long a = src0 + r / 12;
        const uint32_t pix = (uint32_t)(r % 12);
        pool.key[slot0 + r] = ray_key((uint32_t)a, 0, pix);
        pool.s[slot0 + r] = 0.0;
        pool.tau[slot0 + r] = 0.0;
        pool.N[slot0 + r] = cat_L[a] / 12.0;
    }
}

// ---------------------------------------------------------------------------------------------------
// exp(-x) and 1 - exp(-x) for x >= 0, each to a few ulp (not DEC: tolerance 1e-9).
__device__ __forceinline__ void absorb_fraction(double dtau, double &gone, double &left) {
    gone = -expm1(-dtau);                      // Eq. 1's (1 - e^-dtau), accurate for thin cells
    left = (dtau < 0.5) ? (1.0 - gone) : exp(-dtau);
}

enum { OUT_NONE = 0, OUT_SPLIT = 1, OUT_KILL_TAU = 2, OUT_EXIT = 3, OUT_KILL_LMAX = 4 };

// GEOM: 0 no correction, 1 Eq. 5 only, 3 Eq. 5-6 / 7-8 (neighbour deposit; flags live in the field), 4 squared
template <int GEOM>
__global__ void __launch_bounds__(MARCH_THREADS) march_kernel(const __grid_constant__ MarchArgs A) {
    const LoopState *ls = A.ls;
    const long long batch = ls->batch;
    if (batch == 0) return;
    const int level = ls->level;
    const long long begin = ls->begin;
    const int lane = threadIdx.x & 31;
    const double r2s = A.r2_split[level], Kl = A.K[level];
    const long long sy = A.nx, sz = (long long)A.nx * A.ny;

    unsigned long long n_seg = 0, n_zero = 0;
    unsigned int n_split = 0, n_ktau = 0, n_exit = 0, n_klmax = 0;      // lane 0 accumulates warp totals
    double esc = 0.0, res = 0.0, lost = 0.0;

    const long long stride = (long long)gridDim.x * blockDim.x;
    const long long nround = (batch + stride - 1) / stride;
    for (long long it = 0; it < nround; ++it) {
        const long long r = it * stride + (long long)blockIdx.x * blockDim.x + threadIdx.x;
        const bool valid = r < batch;
        int outcome = OUT_NONE;
        uint64_t key = 0;
        double s = 0.0, tau = 0.0, N = 0.0;
        if (valid) {
            key = A.pool.key[begin + r];
            s = A.pool.s[begin + r];
            tau = A.pool.tau[begin + r];
            N = A.pool.N[begin + r];
            const int4 sc = A.cat_cell[key_src(key)];
            double d0, d1, d2;
            pix2dir(level, key_pix(key), d0, d1, d2);
            // O4: start-of-life cell, source-relative (source at its cell centre)
            double q, fl, inv0, inv1, inv2, sx0, sx1, sx2;
            int o0, o1, o2;
            q = fma(s, d0, 0.5); fl = floor(q); o0 = (int)fl; if (q == fl && d0 < 0.0) o0 -= 1;
            q = fma(s, d1, 0.5); fl = floor(q); o1 = (int)fl; if (q == fl && d1 < 0.0) o1 -= 1;
            q = fma(s, d2, 0.5); fl = floor(q); o2 = (int)fl; if (q == fl && d2 < 0.0) o2 -= 1;
            const int st0 = d0 > 0.0 ? 1 : -1, st1 = d1 > 0.0 ? 1 : -1, st2 = d2 > 0.0 ? 1 : -1;
            const int up0 = d0 > 0.0 ? 1 : 0, up1 = d1 > 0.0 ? 1 : 0, up2 = d2 > 0.0 ? 1 : 0;
            if (d0 == 0.0) { inv0 = 0.0; sx0 = CUDART_INF; } else { inv0 = 1.0 / d0; sx0 = ((double)(o0 + up0) - 0.5) * inv0; }
            if (d1 == 0.0) { inv1 = 0.0; sx1 = CUDART_INF; } else { inv1 = 1.0 / d1; sx1 = ((double)(o1 + up1) - 0.5) * inv1; }
            if (d2 == 0.0) { inv2 = 0.0; sx2 = CUDART_INF; } else { inv2 = 1.0 / d2; sx2 = ((double)(o2 + up2) - 0.5) * inv2; }
            int ci = sc.x + o0, cj = sc.y + o1, ck = sc.z + o2;
            if ((unsigned)ci >= (unsigned)A.nx || (unsigned)cj >= (unsigned)A.ny || (unsigned)ck >= (unsigned)A.nz) {
                outcome = OUT_EXIT;
            } else if (tau >= A.tau_max) {
                outcome = OUT_KILL_TAU;
            } else if (level >= A.level_max) {
                outcome = OUT_KILL_LMAX;
            } else {
                long long c = ((long long)ck * A.ny + cj) * A.nx + ci;
                for (;;) {
                    if (tau >= A.tau_max) { outcome = OUT_KILL_TAU; break; }       // 1. filter
                    if (s * s > r2s) { outcome = OUT_SPLIT; break; }               // 3. Eq. 4
                    // 4. one cell
                    int ax = 0;
                    double s_exit = sx0;
                    if (sx1 < s_exit) { s_exit = sx1; ax = 1; }
                    if (sx2 < s_exit) { s_exit = sx2; ax = 2; }
                    double ds = s_exit - s;
                    if (!(ds > 0.0)) ds = 0.0;
                    if (ds > 0.0) {
                        ++n_seg;
                        const double a_c = fabs(__ldg(A.absorber + c));
                        const double dtau = (a_c * A.sdx) * ds;
                        double gone, left;
                        absorb_fraction(dtau, gone, left);
                        const double dN = N * gone;
                        if (dN > 0.0) {
                            double fc = 1.0;
                            long long cn = -1;
                            if (GEOM != 0) {
                                const double s_m = s + 0.5 * ds;
                                double m0 = fma(s_m, d0, 0.5) - (double)o0;
                                double m1 = fma(s_m, d1, 0.5) - (double)o1;
                                double m2 = fma(s_m, d2, 0.5) - (double)o2;
                                m0 = m0 < 0.0 ? 0.0 : (m0 > 1.0 ? 1.0 : m0);
                                m1 = m1 < 0.0 ? 0.0 : (m1 > 1.0 ? 1.0 : m1);
                                m2 = m2 < 0.0 ? 0.0 : (m2 > 1.0 ? 1.0 : m2);
                                double de = m0; int face = 0;                      // first minimum, order x-,x+,y-,y+,z-,z+
                                double t = 1.0 - m0; if (t < de) { de = t; face = 1; }
                                if (m1 < de) { de = m1; face = 2; }
                                t = 1.0 - m1; if (t < de) { de = t; face = 3; }
                                if (m2 < de) { de = m2; face = 4; }
                                t = 1.0 - m2; if (t < de) { de = t; face = 5; }
                                const double l_pix = s_m * Kl;
                                if (de < 0.5 * l_pix) {                            // Eq. 5 / 7, first condition
                                    if (GEOM == 1) fc = 0.5 + de / l_pix;
                                    else if (GEOM == 4) { fc = 0.5 + de / l_pix; fc = fc * fc; }
                                    else {
                                        const int fa = face >> 1, dir = (face & 1) ? 1 : -1;
                                        const int ni = ci + (fa == 0 ? dir : 0), nj = cj + (fa == 1 ? dir : 0),
                                                  nk = ck + (fa == 2 ? dir : 0);
                                        if ((unsigned)ni < (unsigned)A.nx && (unsigned)nj < (unsigned)A.ny &&
                                            (unsigned)nk < (unsigned)A.nz) {
                                            const long long cq = c + (fa == 0 ? dir : (fa == 1 ? dir * sy : dir * sz));
                                            const double a_n = __ldg(A.absorber + cq);   // > 0: absorber present and n_H >= n_th
                                            if (a_n > 0.0) { fc = 0.5 + de / l_pix; cn = cq; }
                                        }
                                    }
                                }
                            }
                            atomicAdd(A.acc + c, fc * dN);
                            if (GEOM == 3) {
                                if (cn >= 0) atomicAdd(A.acc + cn, (1.0 - fc) * dN);
                            } else if (GEOM == 1 || GEOM == 4) {
                                lost += (1.0 - fc) * dN;
                            }
                        }
                        N = N * left;
                        tau = tau + dtau;
                    } else {
                        ++n_zero;
                    }
                    s = s_exit;
                    if (ax == 0) { o0 += st0; ci += st0; c += st0; sx0 = ((double)(o0 + up0) - 0.5) * inv0;
                                   if ((unsigned)ci >= (unsigned)A.nx) { outcome = OUT_EXIT; break; } }
                    else if (ax == 1) { o1 += st1; cj += st1; c += st1 * sy; sx1 = ((double)(o1 + up1) - 0.5) * inv1;
                                   if ((unsigned)cj >= (unsigned)A.ny) { outcome = OUT_EXIT; break; } }
                    else { o2 += st2; ck += st2; c += st2 * sz; sx2 = ((double)(o2 + up2) - 0.5) * inv2;
                                   if ((unsigned)ck >= (unsigned)A.nz) { outcome = OUT_EXIT; break; } }
                }
            }
            if (outcome == OUT_EXIT) esc += N;
            else if (outcome == OUT_KILL_TAU || outcome == OUT_KILL_LMAX) res += N;
        }
        // warp-converged epilogue: counters and child allocation
        const unsigned m_split = __ballot_sync(0xffffffffu, outcome == OUT_SPLIT);
        const unsigned m_ktau = __ballot_sync(0xffffffffu, outcome == OUT_KILL_TAU);
        const unsigned m_exit = __ballot_sync(0xffffffffu, outcome == OUT_EXIT);
        const unsigned m_klmax = __ballot_sync(0xffffffffu, outcome == OUT_KILL_LMAX);
        if (lane == 0) {
            n_split += __popc(m_split); n_ktau += __popc(m_ktau); n_exit += __popc(m_exit); n_klmax += __popc(m_klmax);
        }
        if (m_split) {
            long long base = 0;
            const int nsp = __popc(m_split);
            if (lane == 0) base = atomicAdd((unsigned long long *)&A.ls->count[level + 1], (unsigned long long)(4 * nsp));
            base = __shfl_sync(0xffffffffu, base, 0);
            if (base + 4 * nsp > A.pool.cap[level + 1]) {
                if (lane == 0) A.ls->overflow = 1;
            } else if (outcome == OUT_SPLIT) {
                const long long w = A.pool.off[level + 1] + base + 4 * __popc(m_split & ((1u << lane) - 1u));
                const uint32_t src = key_src(key), p4 = 4u * key_pix(key);
                const double Nc = N * 0.25;                                      // L shared evenly
#pragma unroll
                for (int k = 0; k < 4; ++k) {
                    A.pool.key[w + k] = ray_key(src, level + 1, p4 + k);
                    A.pool.s[w + k] = s;
                    A.pool.tau[w + k] = tau;
                    A.pool.N[w + k] = Nc;
                }
            }
        }
    }
    // flush per-thread / per-warp tallies
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) {
        n_seg += __shfl_xor_sync(0xffffffffu, n_seg, o);
        n_zero += __shfl_xor_sync(0xffffffffu, n_zero, o);
        esc += __shfl_xor_sync(0xffffffffu, esc, o);
        res += __shfl_xor_sync(0xffffffffu, res, o);
        lost += __shfl_xor_sync(0xffffffffu, lost, o);
    }
    if (lane == 0) {
        DevStats *ds = A.ds;
        if (n_seg) atomicAdd(&ds->segments, n_seg);
        if (n_zero) atomicAdd(&ds->zero_len, n_zero);
        if (n_split) atomicAdd(&ds->split[level], (unsigned long long)n_split);
        if (n_ktau) atomicAdd(&ds->killed_tau[level], (unsigned long long)n_ktau);
        if (n_exit) atomicAdd(&ds->exited[level], (unsigned long long)n_exit);
        if (n_klmax) atomicAdd(&ds->killed_lmax[level], (unsigned long long)n_klmax);
        if (esc != 0.0) atomicAdd(&ds->escaped, esc);
        if (res != 0.0) atomicAdd(&ds->residual, res);
        if (lost != 0.0) atomicAdd(&ds->lost, lost);
    }
}

// ---------------------------------------------------------------------------------------------------
// Field preparation (set_fields): absorber a = n_H x_HI in fp64 (reading R1), with the
// sign bit carrying Eq. 7-8's "n_H < n_th" so that the march reads ONE value per
// cell.  Also the per-block partial sums of the ionised fraction 1 - x_HI for automerge.
template <typename T>
__global__ void prep_fields_kernel(const T *__restrict__ nH, const T *__restrict__ xHI, double *__restrict__ a,
                                   long long ncell, double n_th, int use_flag, double *__restrict__ partial) {
    __shared__ double sh[256];
    double acc = 0.0;
    for (long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x; i < ncell;
         i += (long long)gridDim.x * blockDim.x) {
        const double n = (double)nH[i], x = (double)xHI[i];
        double v = n * x;
        if (use_flag && !(n >= n_th)) v = -v;
        a[i] = v;
        acc += 1.0 - x;
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
// per-block partial sums of the deposited photons for the budget.
__global__ void finalise_kernel(double *__restrict__ gamma, double *__restrict__ heat,
                                const double *__restrict__ absorber, long long ncell, double V, double e_excess,
                                double *__restrict__ partial) {
    __shared__ double sh[256];
    double acc = 0.0;
    for (long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x; i < ncell;
         i += (long long)gridDim.x * blockDim.x) {
        const double ph = gamma[i];
        acc += ph;
        if (ph != 0.0) {
            gamma[i] = ph / (fabs(absorber[i]) * V);
            if (heat) heat[i] = e_excess * ph / V;
        } else if (heat) {
            heat[i] = 0.0;
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

__global__ void pix2dir_kernel(int level, long long pix0, long long n, double *out) {
    const long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n) return;
    double x, y, z;
    pix2dir(level, (uint32_t)(pix0 + i), x, y, z);
    out[3 * i] = x; out[3 * i + 1] = y; out[3 * i + 2] = z;
}

}  // namespace nyxrt
