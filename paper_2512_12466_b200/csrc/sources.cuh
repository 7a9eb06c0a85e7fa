// The source pass on the device (rows a1-a3): snap + dedup + sort, MAX_RADIUS and
// MERGE_SOURCES of Alg. 3 (text 313-333).  The paper runs this on the host I/O rank
// over all pairs; here the pair search is binned by cell and the union-find is lock-free, which gives
// the same connected components.  Sums that later steer rounding (dedup flux, centroid) are sequential
// in catalogue order, as DESIGN.md's DEC list requires.
#pragma once
#include <stdint.h>

#include "healpix.cuh"

namespace nyxrt {

struct GridDims { int nx, ny, nz; int periodic; };

// periodic box: index into [0, n); minimum-image difference in
// [-n/2, n/2), the tie n/2 going to -n/2 (reading R31)
__device__ __forceinline__ long long wrap_idx(long long i, long long n) {
    i %= n;
    return i < 0 ? i + n : i;
}
__device__ __forceinline__ long long min_image(long long d, long long n) {
    d = wrap_idx(d, n);
    return (2 * d >= n) ? d - n : d;
}

// key = linear cell index, or -1 and *bad = 1 if the source is outside the box / L invalid (reading R2)
__global__ void snap_kernel(const double *__restrict__ pos, const double *__restrict__ L, long long n, GridDims g,
                            double lo0, double lo1, double lo2, double unit, double dx,
                            long long *__restrict__ key, int *bad) {
    const long long a = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (a >= n) return;
    const double u0 = (pos[3 * a] - lo0) * unit / dx, u1 = (pos[3 * a + 1] - lo1) * unit / dx,
                 u2 = (pos[3 * a + 2] - lo2) * unit / dx;
    const double l = L[a];
    bool ok = (l >= 0.0) && !isinf(l);
    ok = ok && (u0 >= 0.0) && (u0 < (double)g.nx) && (u1 >= 0.0) && (u1 < (double)g.ny) && (u2 >= 0.0) &&
         (u2 < (double)g.nz);
    long long k = -1;
    if (ok) {
        const long long i = (long long)floor(u0), j = (long long)floor(u1), kk = (long long)floor(u2);
        k = (kk * g.ny + j) * g.nx + i;
    } else {
        *bad = 1;
    }
    key[a] = k;
}

__global__ void head_flags_kernel(const long long *__restrict__ key, long long n, int *__restrict__ flag) {
    const long long t = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (t >= n) return;
    flag[t] = (t == 0 || key[t] != key[t - 1]) ? 1 : 0;
}

// one thread per run of equal keys: flux summed in input order (the sort is stable)
__global__ void dedup_kernel(const long long *__restrict__ key, const int *__restrict__ idx,
                             const int *__restrict__ flag, const int *__restrict__ gid_incl, long long n,
                             const double *__restrict__ L, GridDims g, int4 *__restrict__ out_cell,
                             double *__restrict__ out_L, long long *__restrict__ out_key) {
    const long long t = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (t >= n || !flag[t]) return;
    const long long k = key[t];
    double sum = 0.0;
    for (long long u = t; u < n && key[u] == k; ++u) sum = sum + L[idx[u]];
    const int gid = gid_incl[t] - 1;
    const int i = (int)(k % g.nx), j = (int)((k / g.nx) % g.ny), kk = (int)(k / ((long long)g.nx * g.ny));
    out_cell[gid] = make_int4(i, j, kk, 0);
    out_L[gid] = sum;
    out_key[gid] = k;
}

template <typename T>
__device__ __forceinline__ double ion_frac(const T *xHI, long long c) { return 1.0 - (double)xHI[c]; }

// MAX_RADIUS: one warp per source, lanes share the 12*4^samp_level directions of a shell.
template <typename T>
__global__ void radius_kernel(const int4 *__restrict__ cell, long long n, const T *__restrict__ xHI, GridDims g,
                              const double *__restrict__ dirs, int ndir, double delta_r, double r_max, double x_th,
                              double f_req, int n_min_samples, double *__restrict__ r_out) {
    const long long a = ((long long)blockIdx.x * blockDim.x + threadIdx.x) >> 5;
    const int lane = threadIdx.x & 31;
    if (a >= n) return;
    const int4 c = cell[a];
    const double x0 = ion_frac(xHI, ((long long)c.z * g.ny + c.y) * g.nx + c.x);
    if (x0 < x_th) { if (lane == 0) r_out[a] = 0.0; return; }
    double r = delta_r, res = -1.0;
    while (r <= r_max) {
        int ntot = 0, nion = 0;
        for (int q = lane; q < ndir; q += 32) {
            long long i = c.x + (long long)floor(fma(r, dirs[3 * q], 0.5));
            long long j = c.y + (long long)floor(fma(r, dirs[3 * q + 1], 0.5));
            long long k = c.z + (long long)floor(fma(r, dirs[3 * q + 2], 0.5));
            if (g.periodic) { i = wrap_idx(i, g.nx); j = wrap_idx(j, g.ny); k = wrap_idx(k, g.nz); }
            else if (i < 0 || i >= g.nx || j < 0 || j >= g.ny || k < 0 || k >= g.nz) continue;
            ++ntot;
            if (ion_frac(xHI, (k * g.ny + j) * g.nx + i) >= x_th) ++nion;
        }
        ntot = __reduce_add_sync(0xffffffffu, ntot);
        nion = __reduce_add_sync(0xffffffffu, nion);
        bool pass;
        if (ntot == 0) pass = false;
        else if (ntot < n_min_samples) pass = (nion == ntot);
        else pass = ((double)nion >= f_req * (double)ntot);
        if (!pass) { res = r - delta_r; break; }
        r = r + delta_r;
    }
    if (lane == 0) r_out[a] = (res >= 0.0) ? res : r_max;
}

// ---- union-find, smaller index wins (so the root of a component is its smallest member) -------------
// par[x] <= x always, so following parents strictly descends until a root (par[r] == r).  Reads bypass
// L1 (volatile): other threads hook roots concurrently with atomicCAS.  Two passes: walk to the root, then
// point every node of the walked path at it.  The second pass only rewrites non-roots with one of their
// ancestors and hooking only rewrites roots, so the two never collide; a concurrent hook may make `root`
// a non-root meanwhile, which only means the path is compressed to an ancestor instead of the new root.
__device__ __forceinline__ int uf_find(int *par, int a) {
    volatile int *vp = par;
    int root = a;
    for (int up = vp[root]; up != root; up = vp[root]) root = up;
    while (a != root) {
        const int up = vp[a];
        if (up > root) vp[a] = root;
        a = up < root ? root : up;
    }
    return root;
}

__device__ __forceinline__ void uf_unite(int *par, int a, int b) {
    for (;;) {
        a = uf_find(par, a);
        b = uf_find(par, b);
        if (a == b) return;
        if (a > b) { const int t = a; a = b; b = t; }
        // hook the larger root b under the smaller root a
        const int old = atomicCAS(par + b, b, a);
        if (old == b) return;
    }
}

// n = 1: what the sort, the run heads and their scan would produce
__global__ void single_source_kernel(const long long *key_a, long long *key_b, int *idx_b, int *flag, int *gid) {
    if (threadIdx.x == 0) { key_b[0] = key_a[0]; idx_b[0] = 0; flag[0] = 1; gid[0] = 1; }
}

__global__ void iota_kernel(int *p, long long n) {
    const long long a = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (a < n) p[a] = (int)a;
}

__global__ void bin_kernel(const int4 *__restrict__ cell, long long n, int W, int nbx, int nby,
                           int *__restrict__ bin, int *__restrict__ idx) {
    const long long a = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (a >= n) return;
    const int4 c = cell[a];
    bin[a] = ((c.z / W) * nby + (c.y / W)) * nbx + (c.x / W);
    idx[a] = (int)a;
}

constexpr int BIG_GROUP = 64;             // groups of this many members or more go to collapse_big_kernel

__device__ __forceinline__ long long lower_bound_int(const int *v, long long n, int x) {
    long long lo = 0, hi = n;
    while (lo < hi) {
        const long long mid = (lo + hi) >> 1;
        if (v[mid] < x) lo = mid + 1; else hi = mid;
    }
    return lo;
}

// link test of Alg. 3 (PAPER.md:367-370 with the text's epsilon, 331): integer d^2, fp64 right-hand side
// bins to search along one axis: b-1, b, b+1 inside the box; in a periodic box b-2 .. b+2 wrapped (the last
// bin of an axis may be narrower than W, so a pair across the face can sit two bins apart), without repeats
__device__ __forceinline__ int bin_range(int b, int nb, int periodic, int *out) {
    int m = 0;
    if (!periodic) {
        for (int d = -1; d <= 1; ++d)
            if (b + d >= 0 && b + d < nb) out[m++] = b + d;
        return m;
    }
    for (int d = -2; d <= 2; ++d) {
        const int x = (int)wrap_idx(b + d, nb);
        bool seen = false;
        for (int u = 0; u < m; ++u) seen = seen || out[u] == x;
        if (!seen) out[m++] = x;
    }
    return m;
}

__global__ void link_kernel(const int4 *__restrict__ cell, const double *__restrict__ rad, long long n, int W,
                            int nbx, int nby, int nbz, GridDims g, const int *__restrict__ sbin,
                            const int *__restrict__ sidx, double f_ov, double eps, int *par) {
    const long long a = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (a >= n) return;
    const double ra = rad[a];
    if (!(ra > 0.0)) return;
    const int4 ca = cell[a];
    int lx[5], ly[5], lz[5];
    const int mx = bin_range(ca.x / W, nbx, g.periodic, lx), my = bin_range(ca.y / W, nby, g.periodic, ly),
              mz = bin_range(ca.z / W, nbz, g.periodic, lz);
    for (int uz = 0; uz < mz; ++uz)
        for (int uy = 0; uy < my; ++uy)
            for (int ux = 0; ux < mx; ++ux) {
                const int b = (lz[uz] * nby + ly[uy]) * nbx + lx[ux];
                for (long long t = lower_bound_int(sbin, n, b); t < n && sbin[t] == b; ++t) {
                    const int o = sidx[t];
                    if (o <= a) continue;                                   // each pair once (a < b)
                    const double rb = rad[o];
                    if (!(rb > 0.0)) continue;
                    const int4 cb = cell[o];
                    long long ex = (long long)ca.x - cb.x, ey = (long long)ca.y - cb.y, ez = (long long)ca.z - cb.z;
                    if (g.periodic) { ex = min_image(ex, g.nx); ey = min_image(ey, g.ny); ez = min_image(ez, g.nz); }
                    const long long d2 = ex * ex + ey * ey + ez * ez;
                    const double rs = f_ov * (ra + rb);
                    if ((double)d2 <= rs * rs + eps) uf_unite(par, (int)a, o);
                }
            }
}

__global__ void label_kernel(int *par, long long n, int *__restrict__ label, int *__restrict__ idx) {
    const long long a = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (a >= n) return;
    label[a] = uf_find(par, (int)a);
    idx[a] = (int)a;
}

__global__ void head_flags_int_kernel(const int *__restrict__ key, long long n, int *__restrict__ flag) {
    const long long t = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (t >= n) return;
    flag[t] = (t == 0 || key[t] != key[t - 1]) ? 1 : 0;
}

// members of all groups laid out contiguously in group order (the sort by label is stable, so members keep
// their ascending catalogue order): collapse_kernel then streams them instead of chasing sidx -> cell / L / r
__global__ void gather_members_kernel(const int *__restrict__ sidx, long long n, const int4 *__restrict__ cell,
                                      const double *__restrict__ L, const double *__restrict__ rad,
                                      int4 *__restrict__ m_cell, double *__restrict__ m_L, double *__restrict__ m_r) {
    const long long e = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (e >= n) return;
    const int b = sidx[e];
    m_cell[e] = cell[b];
    m_L[e] = L[b];
    m_r[e] = rad[b];
}

// one thread per group (members = a run of equal labels, ascending catalogue index): flux sum, max
// radius, flux-weighted centroid, round, snap to the nearest member (first on ties) -- PAPER.md:378-387.
// cell / L / rad are the member arrays of gather_members_kernel (indexed like slabel).  The sums are
// sequential in member order (DESIGN.md DEC); a percolating group of 10^5 members is one thread's loop.
__global__ void collapse_kernel(const int *__restrict__ slabel,
                                const int *__restrict__ flag, const int *__restrict__ gid_incl, long long n,
                                const int4 *__restrict__ cell, const double *__restrict__ L,
                                const double *__restrict__ rad, GridDims g, int4 *__restrict__ out_cell,
                                double *__restrict__ out_L, double *__restrict__ out_r,
                                long long *__restrict__ out_key, int *__restrict__ big_list, int *big_n) {
    const long long t = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (t >= n || !flag[t]) return;
    const int lab = slabel[t];
    const long long end = lower_bound_int(slabel, n, lab + 1);       // labels are sorted: the run ends here
    if (end - t >= BIG_GROUP) {                                      // a warp does it (collapse_big_kernel)
        big_list[atomicAdd(big_n, 1)] = (int)t;
        return;
    }
    long long e = t;
    double F = 0.0, R = 0.0, n0 = 0.0, n1 = 0.0, n2 = 0.0;
    const int4 ref = cell[t];                      // periodic: images nearest to the first member
    for (; e < end; ++e) {
        const long long b = e;
        const double l = L[b];
        const int4 c = cell[b];
        long long x0 = c.x, x1 = c.y, x2 = c.z;
        if (g.periodic) {
            x0 = ref.x + min_image(x0 - ref.x, g.nx);
            x1 = ref.y + min_image(x1 - ref.y, g.ny);
            x2 = ref.z + min_image(x2 - ref.z, g.nz);
        }
        F = F + l;
        if (rad[b] > R) R = rad[b];
        n0 = n0 + l * (double)x0;
        n1 = n1 + l * (double)x1;
        n2 = n2 + l * (double)x2;
    }
    int4 oc;
    double oL, oR;
    if (e - t == 1) {
        const long long b = t;
        oc = cell[b]; oL = L[b]; oR = rad[b];
    } else {
        long long r0 = (long long)floor(n0 / F + 0.5), r1 = (long long)floor(n1 / F + 0.5),
                  r2 = (long long)floor(n2 / F + 0.5);
        if (g.periodic) { r0 = wrap_idx(r0, g.nx); r1 = wrap_idx(r1, g.ny); r2 = wrap_idx(r2, g.nz); }
        long long bestd = -1;
        long long best = -1;
        for (long long u = t; u < e; ++u) {
            const int4 c = cell[u];
            long long ex = c.x - r0, ey = c.y - r1, ez = c.z - r2;
            if (g.periodic) { ex = min_image(ex, g.nx); ey = min_image(ey, g.ny); ez = min_image(ez, g.nz); }
            const long long d2 = ex * ex + ey * ey + ez * ez;
            if (best < 0 || d2 < bestd) { best = u; bestd = d2; }
        }
        oc = cell[best]; oL = F; oR = R;
    }
    const int gid = gid_incl[t] - 1;
    out_cell[gid] = oc;
    out_L[gid] = oL;
    out_r[gid] = oR;
    out_key[gid] = ((long long)oc.z * g.ny + oc.y) * g.nx + oc.x;
}

// Large groups (a percolating bubble can hold 10^5 sources): one warp per group.  The sums stay sequential in
// member order (DESIGN.md DEC: they steer a rounding) -- lane 0 adds, the warp only stages 32 members at a time
// in shared memory with coalesced loads; the snap (an integer minimum, first member on ties) is a warp reduction.
constexpr int COLLAPSE_WARPS = 4;
__global__ void __launch_bounds__(32 * COLLAPSE_WARPS)
collapse_big_kernel(const int *__restrict__ slabel, const int *__restrict__ gid_incl, long long n,
                    const int4 *__restrict__ cell, const double *__restrict__ L, const double *__restrict__ rad,
                    GridDims g, int4 *__restrict__ out_cell, double *__restrict__ out_L, double *__restrict__ out_r,
                    long long *__restrict__ out_key, const int *__restrict__ big_list, const int *big_n) {
    __shared__ double sl[COLLAPSE_WARPS][32], sr[COLLAPSE_WARPS][32], s0[COLLAPSE_WARPS][32], s1[COLLAPSE_WARPS][32],
        s2[COLLAPSE_WARPS][32];
    const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
    const int nbig = *big_n;
    for (int w = blockIdx.x * COLLAPSE_WARPS + wid; w < nbig; w += gridDim.x * COLLAPSE_WARPS) {
        const long long t = big_list[w];
        const long long end = lower_bound_int(slabel, n, slabel[t] + 1);
        const int4 ref = cell[t];
        double F = 0.0, R = 0.0, n0 = 0.0, n1 = 0.0, n2 = 0.0;
        for (long long base = t; base < end; base += 32) {
            const long long u = base + lane;
            if (u < end) {
                const int4 c = cell[u];
                long long x0 = c.x, x1 = c.y, x2 = c.z;
                if (g.periodic) {
                    x0 = ref.x + min_image(x0 - ref.x, g.nx);
                    x1 = ref.y + min_image(x1 - ref.y, g.ny);
                    x2 = ref.z + min_image(x2 - ref.z, g.nz);
                }
                sl[wid][lane] = L[u]; sr[wid][lane] = rad[u];
                s0[wid][lane] = (double)x0; s1[wid][lane] = (double)x1; s2[wid][lane] = (double)x2;
            }
            __syncwarp();
            if (lane == 0) {
                const int m = (int)((end - base) < 32 ? (end - base) : 32);
                for (int k = 0; k < m; ++k) {
                    const double l = sl[wid][k];
                    F = F + l;
                    if (sr[wid][k] > R) R = sr[wid][k];
                    n0 = n0 + l * s0[wid][k];
                    n1 = n1 + l * s1[wid][k];
                    n2 = n2 + l * s2[wid][k];
                }
            }
            __syncwarp();
        }
        long long r0 = 0, r1 = 0, r2 = 0;
        if (lane == 0) {
            r0 = (long long)floor(n0 / F + 0.5); r1 = (long long)floor(n1 / F + 0.5); r2 = (long long)floor(n2 / F + 0.5);
            if (g.periodic) { r0 = wrap_idx(r0, g.nx); r1 = wrap_idx(r1, g.ny); r2 = wrap_idx(r2, g.nz); }
        }
        r0 = __shfl_sync(0xffffffffu, r0, 0); r1 = __shfl_sync(0xffffffffu, r1, 0); r2 = __shfl_sync(0xffffffffu, r2, 0);
        long long bestd = 0x7fffffffffffffffll, best = 0x7fffffffffffffffll;
        for (long long u = t + lane; u < end; u += 32) {
            const int4 c = cell[u];
            long long ex = c.x - r0, ey = c.y - r1, ez = c.z - r2;
            if (g.periodic) { ex = min_image(ex, g.nx); ey = min_image(ey, g.ny); ez = min_image(ez, g.nz); }
            const long long d2 = ex * ex + ey * ey + ez * ez;
            if (d2 < bestd) { bestd = d2; best = u; }                  // first minimum of this lane's members
        }
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) {                             // first minimum over the lanes
            const long long od = __shfl_down_sync(0xffffffffu, bestd, o), ou = __shfl_down_sync(0xffffffffu, best, o);
            if (od < bestd || (od == bestd && ou < best)) { bestd = od; best = ou; }
        }
        if (lane == 0) {
            const int gid = gid_incl[t] - 1;
            const int4 oc = cell[best];
            out_cell[gid] = oc;
            out_L[gid] = F;
            out_r[gid] = R;
            out_key[gid] = ((long long)oc.z * g.ny + oc.y) * g.nx + oc.x;
        }
    }
}

// gather a catalogue through a permutation (after the final sort by cell key)
__global__ void gather_catalog_kernel(const int *__restrict__ perm, long long n, const int4 *__restrict__ cell,
                                      const double *__restrict__ L, const double *__restrict__ rad,
                                      int4 *__restrict__ out_cell, double *__restrict__ out_L,
                                      double *__restrict__ out_r) {
    const long long a = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (a >= n) return;
    const int p = perm[a];
    out_cell[a] = cell[p];
    out_L[a] = L[p];
    out_r[a] = rad ? rad[p] : 0.0;
}

__global__ void fill_double_kernel(double *p, long long n, double v) {
    const long long a = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (a < n) p[a] = v;
}

// sum of catalogue fluxes = photons emitted (fixed order: single block, strided then tree)
__global__ void sum_flux_kernel(const double *__restrict__ L, long long n, long long first, long long stride, double *out) {
    __shared__ double sh[256];
    double acc = 0.0;
    for (long long i = first + (long long)threadIdx.x * stride; i < n; i += (long long)blockDim.x * stride) acc += L[i];
    sh[threadIdx.x] = acc;
    __syncthreads();
    for (int o = blockDim.x >> 1; o > 0; o >>= 1) {
        if ((int)threadIdx.x < o) sh[threadIdx.x] += sh[threadIdx.x + o];
        __syncthreads();
    }
    if (threadIdx.x == 0) *out = sh[0];
}

}  // namespace nyxrt
