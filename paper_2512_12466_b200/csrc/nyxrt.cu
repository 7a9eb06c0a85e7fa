// C ABI of the B200-native adaptive ray-tracing step (include/nyxrt.h).  Host orchestration only: every
// step of the path runs in the kernels of march.cuh / sources.cuh (plus CUB radix sort and scan as
// library primitives inside the source pass).
#include <cuda_runtime.h>
#include <math_constants.h>

#include <cmath>
#include <cstdarg>
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <new>

#include <cub/device/device_radix_sort.cuh>
#include <cub/device/device_scan.cuh>

#include "../../include/nyxrt.h"
#include "march.cuh"
#include "sources.cuh"
#include "timestep.cuh"

using namespace nyxrt;

namespace {

constexpr int NPARTIAL = 2048;            // blocks of the grid-wide reductions (prep, finalise)

struct SrcBufs {
    double *pos, *L;                       // input sources
    long long *key_a, *key_b;              // cell keys (unsorted / sorted)
    int *idx_a, *idx_b, *flag, *gid;       // permutation, run heads, run ids
    int *par, *lab_a, *lab_b, *bin_a, *bin_b;
    int4 *cell[2];
    double *L2[2], *r[2];
    int4 *m_cell;                          // group members in group order (collapse)
    double *m_L, *m_r;
    long long *ckey[2];
    int *bad;
    double *dirs;                          // shell sample directions, 12*4^samp_level
    void *cub_tmp;
    size_t cub_bytes;
};

}  // namespace

struct nyxrt_ctx {
    nyxrt_grid g;
    nyxrt_params p;
    char err[512];
    int sm_count, march_blocks, nlev;
    long long ncell;
    // workspace
    void *ws;
    uint64_t ws_bytes;
    long long max_sources, batch_rays;
    int host_staging;
    double *absorber, *acc;                // padded grids (nx+2)(ny+2)(nz+2): absorber field, photon accumulator
    double *partial, *scalars;             // scalars[0] = sum(1-x_HI), [1] = absorbed, [2] = emitted
    long long pcell;                       // padded cell count
    bool idx64;                            // padded grid needs 64-bit cell indices
    RayPool pool;
    LoopState *ls;
    DevStats *ds;
    SrcBufs sb;
    void *st_nH, *st_xHI;
    double *st_gamma, *st_heat;
    // state
    const void *d_nH, *d_xHI;
    bool have_fields, have_sources, have_catalog;
    long long n_src, n_dedup, n_cat;
    unsigned long long n_aux_launches;     // own kernels launched outside the ray loop in this trace
    int cat_sel;                           // which of sb.cell[]/L2[]/r[] holds the final catalogue
    int shard_rank, shard_world;           // source sharding (nyxrt_set_shard); 0 of 1 = everything
    double r2_split[MAXLEV], K[MAXLEV];
    double *d_lut;                         // spectrum table on the device (nyxrt_set_spectrum), or null
    double *d_lut_t;                       // table for thin segments (nyxrt_set_spectrum_thin), or null
    double lut_t_first, lut_t_last, tau_thin;
    int lut_e_lo, lut_e_hi, lut_m;
    long long lut_n;
    double lut_first, lut_last;
    cudaEvent_t ev[4];
    cudaEvent_t tev[4];                    // timestep phases
    cudaEvent_t *mev;                      // pairs of events around every march launch
    long long mev_cap;
    cudaStream_t own_stream;
    // the ray loop as one CUDA-graph launch: WHILE node over sched -> emit -> march (rebuilt when its arguments change)
    cudaGraph_t loop_graph;
    cudaGraphExec_t loop_exec;
    MarchArgs loop_args;
    int loop_rank, loop_world;
    const void *loop_fn;
    cudaGraphNode_t loop_finalise;         // the finalise node: its output pointers are patched when they change
    double *loop_gamma, *loop_heat, *loop_photons;
    LoopState *h_ls;                       // pinned
    LoopState *h_ls_init;                  // pinned: the loop state a trace starts from (read by the graph's copy node)
    DevStats *h_ds;                        // pinned
    double *h_scalars;                     // pinned
};

namespace {

int fail(nyxrt_ctx *c, int code, const char *fmt, ...) {
    if (c) {
        va_list ap;
        va_start(ap, fmt);
        vsnprintf(c->err, sizeof c->err, fmt, ap);
        va_end(ap);
    }
    return code;
}

#define CU(call)                                                                                   \
    do {                                                                                           \
        cudaError_t e_ = (call);                                                                   \
        if (e_ != cudaSuccess)                                                                     \
            return fail(ctx, NYXRT_ECUDA, "%s failed: %s (%s:%d)", #call, cudaGetErrorString(e_), \
                        __FILE__, __LINE__);                                                       \
    } while (0)

inline unsigned blocks_for(long long n, int threads) { return (unsigned)((n + threads - 1) / threads); }

size_t field_elem(const nyxrt_ctx *c) { return c->g.field_dtype ? 4 : 8; }

// bump allocator over the workspace; base == nullptr only measures
struct Bump {
    char *base;
    uint64_t off;
    template <typename T>
    T *take(uint64_t n) {
        off = (off + 255) & ~uint64_t(255);
        T *p = base ? reinterpret_cast<T *>(base + off) : nullptr;
        off += n * sizeof(T);
        return p;
    }
};

size_t cub_temp_bytes(long long n) {
    size_t a = 0, b = 0, c = 0;
    cub::DeviceRadixSort::SortPairs(nullptr, a, (long long *)nullptr, (long long *)nullptr, (int *)nullptr,
                                    (int *)nullptr, (int)n);
    cub::DeviceRadixSort::SortPairs(nullptr, b, (int *)nullptr, (int *)nullptr, (int *)nullptr, (int *)nullptr, (int)n);
    cub::DeviceScan::InclusiveSum(nullptr, c, (int *)nullptr, (int *)nullptr, (int)n);
    size_t m = a > b ? a : b;
    return (m > c ? m : c) + 256;
}

// number of pool levels that can hold rays at all: level l needs s^2 > r2_split[l-1] inside the box
int effective_levels(const nyxrt_ctx *c) {
    const double diag2 = (double)c->g.nx * c->g.nx + (double)c->g.ny * c->g.ny + (double)c->g.nz * c->g.nz;
    int nlev = 1;
    while (nlev <= c->p.level_max && c->r2_split[nlev - 1] < diag2) ++nlev;
    return nlev;
}

// the march's geometry stage runs ahead of its box-exit test: a ray that is leaving may read (never use) up to
// three planes plus one neighbour offset beyond the halo; the absorber field carries this many guard cells on
// both sides, and the cell index type must be able to address them
long long guard_cells(const nyxrt_grid &g) { return 4 * ((long long)(g.nx + 2) * (g.ny + 2) + (g.nx + 2) + 4); }

uint64_t layout(nyxrt_ctx *c, void *base, long long max_sources, long long B, int staging) {
    Bump b{static_cast<char *>(base), 0};
    const long long n = max_sources > 0 ? max_sources : 1;
    // the march's geometry stage runs two cells ahead of its box-exit test: a ray that is leaving may read
    // (never use) up to three planes beyond the halo, so the absorber field has a guard band on both sides
    const long long guard = guard_cells(c->g);
    c->absorber = b.take<double>(c->pcell + 2 * guard);
    if (c->absorber) c->absorber += guard;
    c->acc = b.take<double>(c->pcell);
    c->partial = b.take<double>(NPARTIAL);
    c->scalars = b.take<double>(8);
    c->ls = b.take<LoopState>(1);
    c->ds = b.take<DevStats>(1);
    long long total = 0;
    for (int l = 0; l < MAXLEV; ++l) {
        c->pool.off[l] = total;
        // 2B / 5B bound the rays; the slack holds every warp's partly used child slab
        c->pool.cap[l] = l < c->nlev ? (l == 0 ? 2 * B : 5 * B + (long long)CHILD_SLAB * c->march_blocks * MARCH_WARPS) : 0;
        total += c->pool.cap[l];
    }
    c->pool.key = b.take<uint64_t>(total);
    c->pool.s = b.take<double>(total);
    c->pool.tau = b.take<double>(total);
    c->pool.N = b.take<double>(total);
    SrcBufs &s = c->sb;
    s.pos = b.take<double>(3 * n);
    s.L = b.take<double>(n);
    s.key_a = b.take<long long>(n);
    s.key_b = b.take<long long>(n);
    s.idx_a = b.take<int>(n);
    s.idx_b = b.take<int>(n);
    s.flag = b.take<int>(n);
    s.gid = b.take<int>(n);
    s.par = b.take<int>(n);
    s.lab_a = b.take<int>(n);
    s.lab_b = b.take<int>(n);
    s.bin_a = b.take<int>(n);
    s.bin_b = b.take<int>(n);
    for (int k = 0; k < 2; ++k) {
        s.cell[k] = b.take<int4>(n);
        s.L2[k] = b.take<double>(n);
        s.r[k] = b.take<double>(n);
        s.ckey[k] = b.take<long long>(n);
    }
    s.m_cell = b.take<int4>(n);
    s.m_L = b.take<double>(n);
    s.m_r = b.take<double>(n);
    s.bad = b.take<int>(4);
    s.dirs = b.take<double>(3ull * 12ull << (2 * c->p.samp_level));
    s.cub_bytes = cub_temp_bytes(n);
    s.cub_tmp = b.take<char>(s.cub_bytes);
    if (staging) {
        c->st_nH = b.take<char>(c->ncell * field_elem(c));
        c->st_xHI = b.take<char>(c->ncell * field_elem(c));
        c->st_gamma = b.take<double>(c->ncell);
        c->st_heat = b.take<double>(c->ncell);
    } else {
        c->st_nH = c->st_xHI = nullptr;
        c->st_gamma = c->st_heat = nullptr;
    }
    return ((b.off + 255) & ~uint64_t(255));
}

// default rays per march launch: long batches keep the end-of-launch tail small; the pool is (2 + 5 nlev) B rays
long long default_batch(const nyxrt_ctx *c) {
    return c->ncell >= (1ll << 29) ? (1ll << 23) : (c->ncell >= (1ll << 26) ? (1ll << 22) : (1ll << 21));
}

constexpr size_t MARCH_SMEM = 0;          // the kernel's scratch is static shared memory

template <int GEOM, int LUT>
void launch_march(const MarchArgs &a, bool idx64, bool per, int blocks, cudaStream_t st) {
    if (per) {
        if (idx64) march_kernel<GEOM, long long, true, LUT><<<blocks, MARCH_THREADS, MARCH_SMEM, st>>>(a);
        else march_kernel<GEOM, int, true, LUT><<<blocks, MARCH_THREADS, MARCH_SMEM, st>>>(a);
    } else {
        if (idx64) march_kernel<GEOM, long long, false, LUT><<<blocks, MARCH_THREADS, MARCH_SMEM, st>>>(a);
        else march_kernel<GEOM, int, false, LUT><<<blocks, MARCH_THREADS, MARCH_SMEM, st>>>(a);
    }
}

template <typename K>
cudaError_t setup_kernel(K kern, int *occ) {
    cudaError_t e = cudaFuncSetAttribute(kern, cudaFuncAttributePreferredSharedMemoryCarveout, MARCH_CARVEOUT);
    if (e == cudaSuccess) e = cudaOccupancyMaxActiveBlocksPerMultiprocessor(occ, kern, MARCH_THREADS, MARCH_SMEM);
    return e;
}

template <int GEOM, int LUT>
cudaError_t setup_march(bool idx64, bool per, int *occ) {
    if (per) return idx64 ? setup_kernel(march_kernel<GEOM, long long, true, LUT>, occ) : setup_kernel(march_kernel<GEOM, int, true, LUT>, occ);
    return idx64 ? setup_kernel(march_kernel<GEOM, long long, false, LUT>, occ) : setup_kernel(march_kernel<GEOM, int, false, LUT>, occ);
}

// Q(tau_0) of a black body above the H I threshold (PAPER.md:85-95 with sigma ~ nu^-3, R37/R39), by composite
// Simpson in v = nu_0 / nu on (0, 1]:  int_{x0}^inf B(x) (1 - exp(-tau (x0/x)^3)) dx,  B = x^2 / (e^x - 1), x = x0 / v.
// mode 0: the norm int B dx; 1: Q; 2: T = dQ/dtau_0 = int B (x0/x)^3 exp(-tau (x0/x)^3) dx (R40)
double bb_absorbed(double x0, double tau, int mode) {
    const int N = 40000;
    double sum = 0.0;
    for (int i = 1; i <= N; ++i) {                                          // v = 0: the integrand vanishes
        const double v = (double)i / (double)N;
        const double x = x0 / v;
        double f = x * x * std::exp(-x) / -std::expm1(-x) * (x0 / (v * v));
        if (mode == 1) f *= -std::expm1(-tau * v * v * v);
        if (mode == 2) f *= (v * v * v) * std::exp(-tau * v * v * v);
        sum += (i == N ? 1.0 : ((i & 1) ? 4.0 : 2.0)) * f;
    }
    return sum / (3.0 * (double)N);
}

int geom_template(int mode) { return mode == 2 ? 3 : mode; }

template <int GEOM, int LUT>
const void *march_fn_of(bool idx64, bool per) {
    if (per) return idx64 ? (const void *)march_kernel<GEOM, long long, true, LUT> : (const void *)march_kernel<GEOM, int, true, LUT>;
    return idx64 ? (const void *)march_kernel<GEOM, long long, false, LUT> : (const void *)march_kernel<GEOM, int, false, LUT>;
}

const void *march_fn(int gt, bool idx64, bool per, int lut) {
    switch (gt) {
        case 0: return march_fn_of<0, 0>(idx64, per);
        case 1: return march_fn_of<1, 0>(idx64, per);
        case 4: return march_fn_of<4, 0>(idx64, per);
        default: return lut == 2 ? march_fn_of<3, 2>(idx64, per) : (lut == 1 ? march_fn_of<3, 1>(idx64, per) : march_fn_of<3, 0>(idx64, per));
    }
}

void drop_loop_graph(nyxrt_ctx *c) {
    if (c->loop_exec) cudaGraphExecDestroy(c->loop_exec);
    if (c->loop_graph) cudaGraphDestroy(c->loop_graph);
    c->loop_exec = nullptr;
    c->loop_graph = nullptr;
}

// Everything of a trace after the source pass as ONE graph launch (DESIGN.md rows a4-a9): clear the accumulator and
// the counters, copy the initial loop state, a conditional WHILE node whose body is sched -> emit -> march
// (sched_kernel keeps the condition at "rays or sources are left", cudaGraphSetConditional: the device iterates
// without the host and stops after the first empty round), finalise, and the copies of the counters back to pinned
// host memory.  Kernel arguments are baked into the nodes: the graph is rebuilt when they change (new spectrum
// table, shard, workspace); only the output pointers of finalise are patched in place.
struct FinaliseParams {
    double *gamma, *heat;
    const double *acc, *absorber;
    int nx, ny, nz;
    double V, e_excess;
    int periodic;
    double *photons, *partial;
};

cudaError_t set_finalise_params(nyxrt_ctx *c, cudaGraph_t g, cudaGraphNode_t *node, cudaGraphNode_t dep, double *gamma,
                                double *heat, double *photons) {
    FinaliseParams f{gamma, heat, c->acc, c->absorber, c->g.nx, c->g.ny, c->g.nz, c->g.dx_cm * c->g.dx_cm * c->g.dx_cm,
                     c->p.e_excess_erg, c->g.periodic, photons, c->partial};
    void *p[] = {&f.gamma, &f.heat, &f.acc, &f.absorber, &f.nx, &f.ny, &f.nz, &f.V, &f.e_excess, &f.periodic, &f.photons, &f.partial};
    cudaKernelNodeParams kp;
    memset(&kp, 0, sizeof kp);
    kp.func = (void *)finalise_kernel; kp.gridDim = dim3(NPARTIAL); kp.blockDim = dim3(256); kp.kernelParams = p;
    c->loop_gamma = gamma; c->loop_heat = heat; c->loop_photons = photons;
    if (g) return cudaGraphAddKernelNode(node, g, &dep, 1, &kp);
    return cudaGraphExecKernelNodeSetParams(c->loop_exec, *node, &kp);
}

cudaError_t build_loop_graph(nyxrt_ctx *c, const MarchArgs &a, const void *fn, const double *cat_L, int emit_blocks,
                             double *gamma, double *heat, double *photons) {
    drop_loop_graph(c);
    cudaError_t e = cudaGraphCreate(&c->loop_graph, 0);
    if (e != cudaSuccess) return e;
    cudaGraph_t G = c->loop_graph;
    cudaGraphNode_t n_clear, n_stats, n_state, n_while, n_ev2, n_sum, n_ev3, n_c1, n_c2, n_c3;
    cudaMemsetParams mp;
    memset(&mp, 0, sizeof mp);
    mp.dst = c->acc; mp.value = 0; mp.elementSize = 4; mp.width = (size_t)c->pcell * 2; mp.height = 1; mp.pitch = mp.width * 4;
    if ((e = cudaGraphAddMemsetNode(&n_clear, G, nullptr, 0, &mp)) != cudaSuccess) return e;
    mp.dst = c->ds; mp.width = sizeof(DevStats) / 4; mp.pitch = sizeof(DevStats);
    if ((e = cudaGraphAddMemsetNode(&n_stats, G, &n_clear, 1, &mp)) != cudaSuccess) return e;
    if ((e = cudaGraphAddMemcpyNode1D(&n_state, G, &n_stats, 1, c->ls, c->h_ls_init, sizeof(LoopState), cudaMemcpyHostToDevice)) != cudaSuccess) return e;
    cudaGraphConditionalHandle cond;
    if ((e = cudaGraphConditionalHandleCreate(&cond, G, 1, cudaGraphCondAssignDefault)) != cudaSuccess) return e;
    cudaGraphNodeParams cp = {cudaGraphNodeTypeConditional};
    cp.type = cudaGraphNodeTypeConditional;
    cp.conditional.handle = cond;
    cp.conditional.type = cudaGraphCondTypeWhile;
    cp.conditional.size = 1;
    if ((e = cudaGraphAddNode(&n_while, G, &n_state, 1, &cp)) != cudaSuccess) return e;
    cudaGraph_t body = cp.conditional.phGraph_out[0];
    cudaGraphNode_t n_sched, n_emit, n_march;
    int use_cond = 1, nlev = c->nlev, rank = c->shard_rank, world = c->shard_world;
    LoopState *ls = c->ls;
    DevStats *ds = c->ds;
    RayPool pool = c->pool;
    MarchArgs args = a;
    void *p_sched[] = {&ls, &ds, &pool, &nlev, &cond, &use_cond};
    void *p_emit[] = {&ls, &pool, &cat_L, &rank, &world};
    void *p_march[] = {&args};
    cudaKernelNodeParams kp;
    memset(&kp, 0, sizeof kp);
    kp.func = (void *)sched_kernel; kp.gridDim = dim3(1); kp.blockDim = dim3(32); kp.kernelParams = p_sched;
    if ((e = cudaGraphAddKernelNode(&n_sched, body, nullptr, 0, &kp)) != cudaSuccess) return e;
    kp.func = (void *)emit_kernel; kp.gridDim = dim3(emit_blocks); kp.blockDim = dim3(256); kp.kernelParams = p_emit;
    if ((e = cudaGraphAddKernelNode(&n_emit, body, &n_sched, 1, &kp)) != cudaSuccess) return e;
    kp.func = const_cast<void *>(fn); kp.gridDim = dim3(c->march_blocks); kp.blockDim = dim3(MARCH_THREADS); kp.kernelParams = p_march;
    if ((e = cudaGraphAddKernelNode(&n_march, body, &n_emit, 1, &kp)) != cudaSuccess) return e;
    if ((e = cudaGraphAddEventRecordNode(&n_ev2, G, &n_while, 1, c->ev[2])) != cudaSuccess) return e;
    if ((e = set_finalise_params(c, G, &c->loop_finalise, n_ev2, gamma, heat, photons)) != cudaSuccess) return e;
    double *partial = c->partial, *out = c->scalars + 1;
    int np = NPARTIAL;
    void *p_sum[] = {&partial, &np, &out};
    kp.func = (void *)sum_partials_kernel; kp.gridDim = dim3(1); kp.blockDim = dim3(256); kp.kernelParams = p_sum;
    if ((e = cudaGraphAddKernelNode(&n_sum, G, &c->loop_finalise, 1, &kp)) != cudaSuccess) return e;
    if ((e = cudaGraphAddEventRecordNode(&n_ev3, G, &n_sum, 1, c->ev[3])) != cudaSuccess) return e;
    if ((e = cudaGraphAddMemcpyNode1D(&n_c1, G, &n_ev3, 1, c->h_ds, c->ds, sizeof(DevStats), cudaMemcpyDeviceToHost)) != cudaSuccess) return e;
    if ((e = cudaGraphAddMemcpyNode1D(&n_c2, G, &n_c1, 1, c->h_scalars, c->scalars, 8 * sizeof(double), cudaMemcpyDeviceToHost)) != cudaSuccess) return e;
    if ((e = cudaGraphAddMemcpyNode1D(&n_c3, G, &n_c2, 1, c->h_ls, c->ls, sizeof(LoopState), cudaMemcpyDeviceToHost)) != cudaSuccess) return e;
    if ((e = cudaGraphInstantiate(&c->loop_exec, G, 0)) != cudaSuccess) return e;
    c->loop_args = a;
    c->loop_rank = rank;
    c->loop_world = world;
    c->loop_fn = fn;
    return cudaSuccess;
}

// ---- source pass: dedup + sort, optional radius + merge -------------------------------------------
int source_pass(nyxrt_ctx *ctx, cudaStream_t st, bool do_merge) {
    SrcBufs &s = ctx->sb;
    const long long n = ctx->n_src;
    const GridDims gd{ctx->g.nx, ctx->g.ny, ctx->g.nz, ctx->g.periodic};
    ctx->n_dedup = ctx->n_cat = 0;
    ctx->cat_sel = 0;
    if (n == 0) return NYXRT_OK;
    ctx->n_aux_launches += do_merge ? 16 : 4;     // own kernels below (CUB launches not counted)
    int key_bits = 1;
    while (((long long)1 << key_bits) < ctx->ncell) ++key_bits;
    size_t tb = s.cub_bytes;
    // (a1) stable sort by cell key, run heads, sequential flux sums
    if (n == 1) {
        single_source_kernel<<<1, 32, 0, st>>>(s.key_a, s.key_b, s.idx_b, s.flag, s.gid);   // the sorted order of one source
    } else {
        iota_kernel<<<blocks_for(n, 256), 256, 0, st>>>(s.idx_a, n);
        CU(cub::DeviceRadixSort::SortPairs(s.cub_tmp, tb, s.key_a, s.key_b, s.idx_a, s.idx_b, (int)n, 0, key_bits, st));
        head_flags_kernel<<<blocks_for(n, 256), 256, 0, st>>>(s.key_b, n, s.flag);
        tb = s.cub_bytes;
        CU(cub::DeviceScan::InclusiveSum(s.cub_tmp, tb, s.flag, s.gid, (int)n, st));
    }
    dedup_kernel<<<blocks_for(n, 256), 256, 0, st>>>(s.key_b, s.idx_b, s.flag, s.gid, n, s.L, gd, s.cell[0], s.L2[0],
                                                      s.ckey[0]);
    int nd = 1;                                                    // one source: one catalogue entry, no need to ask
    if (n > 1) {
        CU(cudaMemcpyAsync(&nd, s.gid + (n - 1), sizeof(int), cudaMemcpyDeviceToHost, st));
        CU(cudaStreamSynchronize(st));
    }
    ctx->n_dedup = ctx->n_cat = nd;
    fill_double_kernel<<<blocks_for(nd, 256), 256, 0, st>>>(s.r[0], nd, 0.0);
    if (!do_merge) return NYXRT_OK;
    // (a2) bubble radii
    const int ndir = 12 << (2 * ctx->p.samp_level);
    pix2dir_kernel<<<blocks_for(ndir, 128), 128, 0, st>>>(ctx->p.samp_level, 0, ndir, s.dirs);
    const unsigned rb = blocks_for((long long)nd * 32, 256);
    if (ctx->g.field_dtype)
        radius_kernel<float><<<rb, 256, 0, st>>>(s.cell[0], nd, (const float *)ctx->d_xHI, gd, s.dirs, ndir,
                                                  ctx->p.delta_r, ctx->p.r_max, ctx->p.x_th, ctx->p.f_req,
                                                  ctx->p.n_min_samples, s.r[0]);
    else
        radius_kernel<double><<<rb, 256, 0, st>>>(s.cell[0], nd, (const double *)ctx->d_xHI, gd, s.dirs, ndir,
                                                   ctx->p.delta_r, ctx->p.r_max, ctx->p.x_th, ctx->p.f_req,
                                                   ctx->p.n_min_samples, s.r[0]);
    // (a3) links between overlapping bubbles: bins of width W >= the largest link distance
    const double X = 2.0 * ctx->p.f_ov * ctx->p.r_max;
    long long Wl = (long long)floor(sqrt(X * X + ctx->p.eps)) + 1;
    if (Wl < 1) Wl = 1;
    if (Wl > (1 << 20)) Wl = 1 << 20;
    const int W = (int)Wl;
    const int nbx = (ctx->g.nx + W - 1) / W, nby = (ctx->g.ny + W - 1) / W, nbz = (ctx->g.nz + W - 1) / W;
    int bin_bits = 1;
    while (((long long)1 << bin_bits) < (long long)nbx * nby * nbz) ++bin_bits;
    const unsigned nb = blocks_for(nd, 256);
    bin_kernel<<<nb, 256, 0, st>>>(s.cell[0], nd, W, nbx, nby, s.bin_a, s.idx_a);
    tb = s.cub_bytes;
    CU(cub::DeviceRadixSort::SortPairs(s.cub_tmp, tb, s.bin_a, s.bin_b, s.idx_a, s.idx_b, nd, 0, bin_bits, st));
    iota_kernel<<<nb, 256, 0, st>>>(s.par, nd);
    link_kernel<<<nb, 256, 0, st>>>(s.cell[0], s.r[0], nd, W, nbx, nby, nbz, gd, s.bin_b, s.idx_b, ctx->p.f_ov, ctx->p.eps,
                                    s.par);
    // groups: label = smallest member; members in ascending catalogue order (stable sort by label)
    label_kernel<<<nb, 256, 0, st>>>(s.par, nd, s.lab_a, s.idx_a);
    int lab_bits = 1;
    while (((long long)1 << lab_bits) < nd) ++lab_bits;
    tb = s.cub_bytes;
    CU(cub::DeviceRadixSort::SortPairs(s.cub_tmp, tb, s.lab_a, s.lab_b, s.idx_a, s.idx_b, nd, 0, lab_bits, st));
    head_flags_int_kernel<<<nb, 256, 0, st>>>(s.lab_b, nd, s.flag);
    tb = s.cub_bytes;
    CU(cub::DeviceScan::InclusiveSum(s.cub_tmp, tb, s.flag, s.gid, nd, st));
    gather_members_kernel<<<nb, 256, 0, st>>>(s.idx_b, nd, s.cell[0], s.L2[0], s.r[0], s.m_cell, s.m_L, s.m_r);
    CU(cudaMemsetAsync(s.bad + 1, 0, sizeof(int), st));               // number of large groups
    collapse_kernel<<<nb, 256, 0, st>>>(s.lab_b, s.flag, s.gid, nd, s.m_cell, s.m_L, s.m_r, gd, s.cell[1],
                                        s.L2[1], s.r[1], s.ckey[1], s.bin_a, s.bad + 1);
    collapse_big_kernel<<<ctx->sm_count * 2, 32 * COLLAPSE_WARPS, 0, st>>>(s.lab_b, s.gid, nd, s.m_cell, s.m_L, s.m_r, gd,
                                                                          s.cell[1], s.L2[1], s.r[1], s.ckey[1], s.bin_a,
                                                                          s.bad + 1);
    int nm = 1;
    if (nd > 1) {
        CU(cudaMemcpyAsync(&nm, s.gid + (nd - 1), sizeof(int), cudaMemcpyDeviceToHost, st));
        CU(cudaStreamSynchronize(st));
    }
    // final sort by cell key; keys are unique
    iota_kernel<<<blocks_for(nm, 256), 256, 0, st>>>(s.idx_a, nm);
    tb = s.cub_bytes;
    CU(cub::DeviceRadixSort::SortPairs(s.cub_tmp, tb, s.ckey[1], s.ckey[0], s.idx_a, s.idx_b, nm, 0, key_bits, st));
    gather_catalog_kernel<<<blocks_for(nm, 256), 256, 0, st>>>(s.idx_b, nm, s.cell[1], s.L2[1], s.r[1], s.cell[0],
                                                                s.L2[0], s.r[0]);
    ctx->n_cat = nm;
    CU(cudaGetLastError());
    return NYXRT_OK;
}

}  // namespace

// =================================================================================================
extern "C" {

int nyxrt_version(void) { return 100; }
int nyxrt_sizeof_grid(void) { return (int)sizeof(nyxrt_grid); }
int nyxrt_sizeof_params(void) { return (int)sizeof(nyxrt_params); }
int nyxrt_sizeof_stats(void) { return (int)sizeof(nyxrt_stats); }
int nyxrt_sizeof_ode(void) { return (int)sizeof(nyxrt_ode); }
int nyxrt_sizeof_tstats(void) { return (int)sizeof(nyxrt_tstats); }

const char *nyxrt_last_error(const nyxrt_ctx *ctx) { return ctx ? ctx->err : "null context"; }

int nyxrt_create(const nyxrt_grid *grid, const nyxrt_params *params, nyxrt_ctx **out) {
    if (!grid || !params || !out) return NYXRT_EINVAL;
    *out = nullptr;
    const nyxrt_grid &g = *grid;
    const nyxrt_params &p = *params;
    if (g.nx < 1 || g.ny < 1 || g.nz < 1 || g.nx > (1 << 20) || g.ny > (1 << 20) || g.nz > (1 << 20)) return NYXRT_EINVAL;
    if ((long long)g.nx * g.ny * g.nz >= ((long long)1 << 40)) return NYXRT_EINVAL;
    if (g.field_dtype != 0 && g.field_dtype != 1) return NYXRT_EINVAL;
    if (!(g.dx_cm > 0.0) || !(g.pos_unit_cm > 0.0) || (g.periodic != 0 && g.periodic != 1)) return NYXRT_EINVAL;
    if (!(p.sigma_cm2 > 0.0) || !(p.n_min_ray > 0.0) || !(p.tau_max > 0.0)) return NYXRT_EINVAL;
    if (p.level_max < 0 || p.level_max > 13 || p.geom_mode < 0 || p.geom_mode > 4) return NYXRT_EINVAL;
    if (p.merge < 0 || p.merge > 2 || p.samp_level < 0 || p.samp_level > 8 || !(p.delta_r > 0.0)) return NYXRT_EINVAL;
    if (!(p.r_max >= 0.0) || !(p.f_ov >= 0.0)) return NYXRT_EINVAL;
    nyxrt_ctx *ctx = new (std::nothrow) nyxrt_ctx();
    if (!ctx) return NYXRT_ENOMEM;
    memset(ctx, 0, sizeof *ctx);
    ctx->g = g;
    ctx->p = p;
    ctx->ncell = (long long)g.nx * g.ny * g.nz;
    ctx->shard_rank = 0;
    ctx->shard_world = 1;
    ctx->pcell = (long long)(g.nx + 2) * (g.ny + 2) * (g.nz + 2);
    ctx->idx64 = ctx->pcell + guard_cells(g) >= (1ll << 31);      // the guard band must be addressable too
    const double PI = 0x1.921fb54442d18p+1;
    for (int l = 0; l < MAXLEV; ++l) {
        ctx->r2_split[l] = std::ldexp(3.0 / (PI * p.n_min_ray), 2 * l);   // Eq. 4
        ctx->K[l] = std::ldexp(std::sqrt(PI / 3.0), -l);                  // sqrt(4 pi / (12 4^l))
    }
    ctx->nlev = effective_levels(ctx);
    cudaError_t e = cudaSetDevice(g.device);
    cudaDeviceProp prop;
    if (e == cudaSuccess) e = cudaGetDeviceProperties(&prop, g.device);
    if (e == cudaSuccess) e = cudaStreamCreateWithFlags(&ctx->own_stream, cudaStreamNonBlocking);
    for (int k = 0; k < 4 && e == cudaSuccess; ++k) e = cudaEventCreate(&ctx->ev[k]);
    for (int k = 0; k < 4 && e == cudaSuccess; ++k) e = cudaEventCreate(&ctx->tev[k]);
    if (e == cudaSuccess) e = cudaMallocHost(&ctx->h_ls, sizeof(LoopState));
    if (e == cudaSuccess) e = cudaMallocHost(&ctx->h_ls_init, sizeof(LoopState));
    if (e == cudaSuccess) e = cudaMallocHost(&ctx->h_ds, sizeof(DevStats));
    if (e == cudaSuccess) e = cudaMallocHost(&ctx->h_scalars, 8 * sizeof(double));
    int occ = 0;
    if (e == cudaSuccess) {
        switch (geom_template(p.geom_mode)) {
            case 0: e = setup_march<0, 0>(ctx->idx64, g.periodic != 0, &occ); break;
            case 1: e = setup_march<1, 0>(ctx->idx64, g.periodic != 0, &occ); break;
            case 4: e = setup_march<4, 0>(ctx->idx64, g.periodic != 0, &occ); break;
            default: {
                int occ_lut = 0, occ_thin = 0;
                e = setup_march<3, 1>(ctx->idx64, g.periodic != 0, &occ_lut);
                if (e == cudaSuccess) e = setup_march<3, 2>(ctx->idx64, g.periodic != 0, &occ_thin);
                if (e == cudaSuccess) e = setup_march<3, 0>(ctx->idx64, g.periodic != 0, &occ);
                if (occ_lut < occ) occ = occ_lut;
                if (occ_thin < occ) occ = occ_thin;
                break;
            }
        }
    }
    if (e != cudaSuccess) {
        // no CUDA device / wrong architecture: there is no fallback
        nyxrt_destroy(ctx);
        return NYXRT_ECUDA;
    }
    ctx->sm_count = prop.multiProcessorCount;
    ctx->march_blocks = ctx->sm_count * (occ > 0 ? occ : 1);
    *out = ctx;
    return NYXRT_OK;
}

void nyxrt_destroy(nyxrt_ctx *ctx) {
    if (!ctx) return;
    drop_loop_graph(ctx);
    for (long long k = 0; k < ctx->mev_cap; ++k) cudaEventDestroy(ctx->mev[k]);
    free(ctx->mev);
    for (int k = 0; k < 4; ++k)
        if (ctx->ev[k]) cudaEventDestroy(ctx->ev[k]);
    for (int k = 0; k < 4; ++k)
        if (ctx->tev[k]) cudaEventDestroy(ctx->tev[k]);
    if (ctx->d_lut) cudaFree(ctx->d_lut);
    if (ctx->d_lut_t) cudaFree(ctx->d_lut_t);
    if (ctx->own_stream) cudaStreamDestroy(ctx->own_stream);
    if (ctx->h_ls) cudaFreeHost(ctx->h_ls);
    if (ctx->h_ls_init) cudaFreeHost(ctx->h_ls_init);
    if (ctx->h_ds) cudaFreeHost(ctx->h_ds);
    if (ctx->h_scalars) cudaFreeHost(ctx->h_scalars);
    delete ctx;
}

int nyxrt_workspace_bytes(const nyxrt_ctx *cctx, int64_t max_sources, int64_t batch_rays, int32_t host_staging,
                          uint64_t *bytes) {
    if (!cctx || !bytes || max_sources < 0 || batch_rays < 0 || max_sources >= (1ll << 30)) return NYXRT_EINVAL;
    const long long B = batch_rays ? batch_rays : default_batch(cctx);
    if (B < 32) return NYXRT_EINVAL;
    nyxrt_ctx scratch = *cctx;                    // a pure query: the layout is laid out on a copy
    *bytes = layout(&scratch, nullptr, max_sources, B, host_staging);
    return NYXRT_OK;
}

int nyxrt_set_workspace(nyxrt_ctx *ctx, void *d_ws, uint64_t bytes, int64_t max_sources, int64_t batch_rays,
                        int32_t host_staging) {
    if (!ctx) return NYXRT_EINVAL;
    if (!d_ws || ((uintptr_t)d_ws & 255) || max_sources < 0 || batch_rays < 0 || max_sources >= (1ll << 30))
        return fail(ctx, NYXRT_EINVAL, "set_workspace: bad argument (pointer must be 256-byte aligned)");
    const long long B = batch_rays ? batch_rays : default_batch(ctx);
    if (B < 32) return fail(ctx, NYXRT_EINVAL, "set_workspace: batch_rays must be >= 32");
    ctx->ws = nullptr;
    nyxrt_ctx scratch = *ctx;
    const uint64_t need = layout(&scratch, nullptr, max_sources, B, host_staging);
    if (bytes < need) return fail(ctx, NYXRT_ENOMEM, "set_workspace: %llu bytes given, %llu needed",
                                  (unsigned long long)bytes, (unsigned long long)need);
    layout(ctx, d_ws, max_sources, B, host_staging);
    ctx->ws = d_ws;
    ctx->ws_bytes = bytes;
    ctx->max_sources = max_sources;
    ctx->batch_rays = B;
    ctx->host_staging = host_staging;
    ctx->have_fields = ctx->have_sources = ctx->have_catalog = false;
    return NYXRT_OK;
}

int nyxrt_set_fields(nyxrt_ctx *ctx, const void *d_nH, const void *d_xHI, void *cuda_stream) {
    if (!ctx) return NYXRT_EINVAL;
    if (!d_nH || !d_xHI) return fail(ctx, NYXRT_EINVAL, "set_fields: null field pointer");
    if (!ctx->ws) return fail(ctx, NYXRT_ESTATE, "set_fields: no workspace");
    cudaStream_t st = (cudaStream_t)cuda_stream;
    CU(cudaSetDevice(ctx->g.device));
    const int use_flag = ctx->p.geom_mode == 3;
    if (ctx->g.field_dtype)
        prep_fields_kernel<float><<<NPARTIAL, 256, 0, st>>>((const float *)d_nH, (const float *)d_xHI, ctx->absorber,
                                                            ctx->g.nx, ctx->g.ny, ctx->g.nz, ctx->p.n_th, use_flag,
                                                            ctx->g.periodic, ctx->partial);
    else
        prep_fields_kernel<double><<<NPARTIAL, 256, 0, st>>>((const double *)d_nH, (const double *)d_xHI, ctx->absorber,
                                                             ctx->g.nx, ctx->g.ny, ctx->g.nz, ctx->p.n_th, use_flag,
                                                             ctx->g.periodic, ctx->partial);
    sum_partials_kernel<<<1, 256, 0, st>>>(ctx->partial, NPARTIAL, ctx->scalars + 0);
    CU(cudaGetLastError());
    ctx->d_nH = d_nH;
    ctx->d_xHI = d_xHI;
    ctx->have_fields = true;
    return NYXRT_OK;
}

int nyxrt_set_sources(nyxrt_ctx *ctx, int64_t n, const double *pos, const double *L, void *cuda_stream) {
    if (!ctx) return NYXRT_EINVAL;
    ctx->have_sources = false;
    ctx->have_catalog = false;
    if (n < 0 || (n > 0 && (!pos || !L))) return fail(ctx, NYXRT_EINVAL, "set_sources: bad argument");
    if (!ctx->ws) return fail(ctx, NYXRT_ESTATE, "set_sources: no workspace");
    if (n > ctx->max_sources) return fail(ctx, NYXRT_ENOMEM, "set_sources: %lld sources, workspace sized for %lld",
                                          (long long)n, ctx->max_sources);
    cudaStream_t st = (cudaStream_t)cuda_stream;
    CU(cudaSetDevice(ctx->g.device));
    ctx->n_src = n;
    if (n > 0) {
        SrcBufs &s = ctx->sb;
        CU(cudaMemcpyAsync(s.pos, pos, 3 * n * sizeof(double), cudaMemcpyHostToDevice, st));
        CU(cudaMemcpyAsync(s.L, L, n * sizeof(double), cudaMemcpyHostToDevice, st));
        CU(cudaMemsetAsync(s.bad, 0, sizeof(int), st));
        const GridDims gd{ctx->g.nx, ctx->g.ny, ctx->g.nz, ctx->g.periodic};
        snap_kernel<<<blocks_for(n, 256), 256, 0, st>>>(s.pos, s.L, n, gd, ctx->g.box_lo[0], ctx->g.box_lo[1],
                                                         ctx->g.box_lo[2], ctx->g.pos_unit_cm, ctx->g.dx_cm, s.key_a,
                                                         s.bad);
        int bad = 0;
        CU(cudaMemcpyAsync(&bad, s.bad, sizeof(int), cudaMemcpyDeviceToHost, st));
        CU(cudaStreamSynchronize(st));
        if (bad) {
            ctx->n_src = 0;
            return fail(ctx, NYXRT_EINVAL, "set_sources: a source lies outside the box or has an invalid luminosity");
        }
    }
    ctx->have_sources = true;
    return NYXRT_OK;
}

static int run_trace(nyxrt_ctx *ctx, double *d_gamma, double *d_heat, double *d_photons, nyxrt_stats *hs, void *cuda_stream) {
    if (!ctx) return NYXRT_EINVAL;
    if (!d_gamma && !d_photons) return fail(ctx, NYXRT_EINVAL, "trace: null output");
    if (!ctx->ws || !ctx->have_fields || !ctx->have_sources)
        return fail(ctx, NYXRT_ESTATE, "trace: workspace, fields and sources must be set first");
    cudaStream_t st = (cudaStream_t)cuda_stream;
    CU(cudaSetDevice(ctx->g.device));
    CU(cudaEventRecord(ctx->ev[0], st));
    // ---- sources ----
    bool do_merge = ctx->p.merge == 1;
    if (ctx->p.merge == 2) {
        CU(cudaMemcpyAsync(ctx->h_scalars, ctx->scalars, sizeof(double), cudaMemcpyDeviceToHost, st));
        CU(cudaStreamSynchronize(st));
        do_merge = ctx->h_scalars[0] / (double)ctx->ncell > ctx->p.automerge_xmean;
    }
    ctx->n_aux_launches = 3;                      // sum_flux, finalise, sum_partials
    int rc = source_pass(ctx, st, do_merge);
    if (rc) return rc;
    ctx->have_catalog = true;
    const SrcBufs &s = ctx->sb;
    sum_flux_kernel<<<1, 256, 0, st>>>(s.L2[0], ctx->n_cat, ctx->shard_rank, ctx->shard_world, ctx->scalars + 2);
    // this shard's sources: catalogue entries rank, rank + world, ... (all of them when world = 1)
    const long long n_local = ctx->n_cat > ctx->shard_rank ? (ctx->n_cat - ctx->shard_rank + ctx->shard_world - 1) / ctx->shard_world : 0;
    CU(cudaEventRecord(ctx->ev[1], st));
    // ---- ray loop ----
    const bool timing = (ctx->p.flags & NYXRT_FLAG_LAUNCH_TIMING) != 0;
    memset(ctx->h_ls_init, 0, sizeof(LoopState));
    ctx->h_ls_init->n_cat = n_local;
    ctx->h_ls_init->batch_rays = ctx->batch_rays;
    if (timing) {
        CU(cudaMemsetAsync(ctx->acc, 0, ctx->pcell * sizeof(double), st));
        CU(cudaMemsetAsync(ctx->ds, 0, sizeof(DevStats), st));
        CU(cudaMemcpyAsync(ctx->ls, ctx->h_ls_init, sizeof(LoopState), cudaMemcpyHostToDevice, st));
    }
    MarchArgs a;
    memset(&a, 0, sizeof a);
    a.absorber = ctx->absorber;
    a.acc = ctx->acc;
    a.cat_cell = s.cell[0];
    a.cat_L = s.L2[0];
    a.pool = ctx->pool;
    a.ls = ctx->ls;
    a.ds = ctx->ds;
    a.nx = ctx->g.nx; a.ny = ctx->g.ny; a.nz = ctx->g.nz;
    a.level_max = ctx->p.level_max;
    a.px = ctx->g.nx + 2;
    a.pxy = (long long)(ctx->g.nx + 2) * (ctx->g.ny + 2);
    a.sdx = ctx->p.sigma_cm2 * ctx->g.dx_cm;
    a.tau_max = ctx->p.tau_max;
    a.s_max = std::sqrt((double)((long long)ctx->g.nx * ctx->g.nx + (long long)ctx->g.ny * ctx->g.ny +
                                 (long long)ctx->g.nz * ctx->g.nz));       // sqrt(3) L_box for a cube
    for (int l = 0; l < MAXLEV; ++l) { a.r2_split[l] = ctx->r2_split[l]; a.K[l] = ctx->K[l]; }
    const bool lut = ctx->d_lut != nullptr;
    if (lut) {
        a.lut_q = ctx->d_lut;
        a.lut_t_lo = std::ldexp(1.0, ctx->lut_e_lo);
        a.lut_t_hi = std::ldexp(1.0, ctx->lut_e_hi);
        a.lut_inv_t_lo = std::ldexp(1.0, -ctx->lut_e_lo);
        a.lut_q_first = ctx->lut_first;
        a.lut_q_last = ctx->lut_last;
        a.lut_fb = 52 - ctx->lut_m;
        a.lut_fscale = std::ldexp(1.0, -a.lut_fb);
        a.lut_fmask = (1ll << a.lut_fb) - 1;
        a.lut_k0 = (long long)(ctx->lut_e_lo + 1023) << ctx->lut_m;
        a.lut_t = ctx->d_lut_t;
        a.lut_t_first = ctx->lut_t_first;
        a.lut_t_last = ctx->lut_t_last;
        a.tau_thin = ctx->tau_thin;
    }
    const int gt = geom_template(ctx->p.geom_mode);
    const int emit_blocks = ctx->sm_count * 4;
    int chunk = 8;
    long long n_launch = 0;
    if (!timing) {
        // production: clear, loop, finalise and the copies back are one graph launch; the host synchronises once
        const void *fn = march_fn(gt, ctx->idx64, ctx->g.periodic != 0, lut ? (ctx->d_lut_t ? 2 : 1) : 0);
        if (!ctx->loop_exec || fn != ctx->loop_fn || ctx->loop_rank != ctx->shard_rank || ctx->loop_world != ctx->shard_world ||
            memcmp(&a, &ctx->loop_args, sizeof a) != 0)
            CU(build_loop_graph(ctx, a, fn, s.L2[0], emit_blocks, d_gamma, d_heat, d_photons));
        else if (d_gamma != ctx->loop_gamma || d_heat != ctx->loop_heat || d_photons != ctx->loop_photons)
            CU(set_finalise_params(ctx, nullptr, &ctx->loop_finalise, nullptr, d_gamma, d_heat, d_photons));
        CU(cudaGraphLaunch(ctx->loop_exec, st));
    }
    for (; timing;) {
        for (int i = 0; i < chunk; ++i) {
            sched_kernel<<<1, 32, 0, st>>>(ctx->ls, ctx->ds, ctx->pool, ctx->nlev, (cudaGraphConditionalHandle)0, 0);
            emit_kernel<<<emit_blocks, 256, 0, st>>>(ctx->ls, ctx->pool, s.L2[0], ctx->shard_rank, ctx->shard_world);
            if (n_launch + 1 > ctx->mev_cap / 2) {                       // grow the event pool
                const long long cap = ctx->mev_cap ? 2 * ctx->mev_cap : 1024;
                cudaEvent_t *m = (cudaEvent_t *)realloc(ctx->mev, cap * sizeof(cudaEvent_t));
                if (!m) return fail(ctx, NYXRT_ENOMEM, "trace: host allocation failed");
                ctx->mev = m;
                for (long long k = ctx->mev_cap; k < cap; ++k) CU(cudaEventCreate(&ctx->mev[k]));
                ctx->mev_cap = cap;
            }
            CU(cudaEventRecord(ctx->mev[2 * n_launch], st));
            switch (gt) {
                case 0: launch_march<0, 0>(a, ctx->idx64, ctx->g.periodic != 0, ctx->march_blocks, st); break;
                case 1: launch_march<1, 0>(a, ctx->idx64, ctx->g.periodic != 0, ctx->march_blocks, st); break;
                case 4: launch_march<4, 0>(a, ctx->idx64, ctx->g.periodic != 0, ctx->march_blocks, st); break;
                default:
                    if (lut && ctx->d_lut_t) launch_march<3, 2>(a, ctx->idx64, ctx->g.periodic != 0, ctx->march_blocks, st);
                    else if (lut) launch_march<3, 1>(a, ctx->idx64, ctx->g.periodic != 0, ctx->march_blocks, st);
                    else launch_march<3, 0>(a, ctx->idx64, ctx->g.periodic != 0, ctx->march_blocks, st);
                    break;
            }
            CU(cudaEventRecord(ctx->mev[2 * n_launch + 1], st));
            ++n_launch;
        }
        CU(cudaMemcpyAsync(ctx->h_ls, ctx->ls, sizeof(LoopState), cudaMemcpyDeviceToHost, st));
        CU(cudaStreamSynchronize(st));
        if (ctx->h_ls->overflow) return fail(ctx, NYXRT_EOVERFLOW, "trace: ray pool overflow at level %d", ctx->h_ls->level + 1);
        if (ctx->h_ls->done) break;
        if (chunk < 256) chunk *= 2;
    }
    if (timing) {
        CU(cudaEventRecord(ctx->ev[2], st));
        // ---- finalise ----
        const double V = ctx->g.dx_cm * ctx->g.dx_cm * ctx->g.dx_cm;
        finalise_kernel<<<NPARTIAL, 256, 0, st>>>(d_gamma, d_heat, ctx->acc, ctx->absorber, ctx->g.nx, ctx->g.ny, ctx->g.nz, V,
                                                  ctx->p.e_excess_erg, ctx->g.periodic, d_photons, ctx->partial);
        sum_partials_kernel<<<1, 256, 0, st>>>(ctx->partial, NPARTIAL, ctx->scalars + 1);
        CU(cudaEventRecord(ctx->ev[3], st));
        CU(cudaMemcpyAsync(ctx->h_ds, ctx->ds, sizeof(DevStats), cudaMemcpyDeviceToHost, st));
        CU(cudaMemcpyAsync(ctx->h_scalars, ctx->scalars, 8 * sizeof(double), cudaMemcpyDeviceToHost, st));
    }
    CU(cudaStreamSynchronize(st));
    CU(cudaGetLastError());
    if (!timing) {
        if (ctx->h_ls->overflow) return fail(ctx, NYXRT_EOVERFLOW, "trace: ray pool overflow at level %d", ctx->h_ls->level + 1);
        n_launch = (long long)ctx->h_ls->iterations + 1;                 // rounds of the WHILE body (the last one is empty)
    }
    if (hs) {
        memset(hs, 0, sizeof *hs);
        const DevStats &d = *ctx->h_ds;
        for (int l = 0; l < MAXLEV; ++l) {
            hs->spawned[l] = d.spawned[l] - d.holes[l]; hs->split[l] = d.split[l]; hs->killed_tau[l] = d.killed_tau[l];
            hs->exited[l] = d.exited[l]; hs->killed_lmax[l] = d.killed_lmax[l];
        }
        hs->segments = d.segments;
        hs->zero_len_segments = d.zero_len;
        hs->neighbour_deposits = d.nbr_deposits;
        hs->n_src_in = (uint64_t)ctx->n_src;
        hs->n_src_dedup = (uint64_t)ctx->n_dedup;
        hs->n_src_merged = (uint64_t)ctx->n_cat;
        hs->iterations = ctx->h_ls->iterations;
        hs->peak_pool_rays = ctx->h_ls->peak_pool;
        hs->photons_emitted = n_local ? ctx->h_scalars[2] : 0.0;
        hs->photons_absorbed = ctx->h_scalars[1];
        hs->photons_escaped = d.escaped;
        hs->photons_residual = d.residual;
        hs->photons_lost = d.lost;
        cudaEventElapsedTime(&hs->ms_sources, ctx->ev[0], ctx->ev[1]);
        cudaEventElapsedTime(&hs->ms_loop, ctx->ev[1], ctx->ev[2]);
        cudaEventElapsedTime(&hs->ms_finalise, ctx->ev[2], ctx->ev[3]);
        cudaEventElapsedTime(&hs->ms_total, ctx->ev[0], ctx->ev[3]);
        double ms = 0.0;
        const long long live = (long long)ctx->h_ls->iterations;       // launches that had a batch
        for (long long k = 0; timing && k < n_launch && k < live; ++k) {
            float t = 0.f;
            cudaEventElapsedTime(&t, ctx->mev[2 * k], ctx->mev[2 * k + 1]);
            ms += t;
        }
        hs->ms_march = (float)ms;
        hs->march_launches = (uint64_t)live;
        hs->kernel_launches = (uint64_t)(3 * n_launch) + ctx->n_aux_launches;
    }
    return NYXRT_OK;
}

int nyxrt_trace(nyxrt_ctx *ctx, double *d_gamma, double *d_heat, nyxrt_stats *hs, void *cuda_stream) {
    if (!ctx) return NYXRT_EINVAL;
    if (!d_gamma) return fail(ctx, NYXRT_EINVAL, "trace: null output");
    if (ctx->shard_world != 1) return fail(ctx, NYXRT_ESTATE, "trace: a shard is set; use trace_photons + finalise");
    return run_trace(ctx, d_gamma, d_heat, nullptr, hs, cuda_stream);
}

int nyxrt_spectrum_nodes(int32_t e_lo, int32_t e_hi, int32_t m, int64_t *n) {
    if (!n || e_lo < -1000 || e_hi > 1000 || e_hi <= e_lo || m < 0 || m > 16) return NYXRT_EINVAL;
    *n = (((int64_t)(e_hi - e_lo)) << m) + 1;
    return *n <= (1ll << 24) ? NYXRT_OK : NYXRT_EINVAL;
}

int nyxrt_spectrum_node_tau(int32_t e_lo, int32_t m, int64_t k, double *tau) {
    if (!tau || m < 0 || m > 16 || k < 0) return NYXRT_EINVAL;
    const int64_t oct = k >> m, sub = k & (((int64_t)1 << m) - 1);
    *tau = std::ldexp(1.0 + (double)sub / (double)((int64_t)1 << m), e_lo + (int)oct);
    return NYXRT_OK;
}

int nyxrt_set_spectrum(nyxrt_ctx *ctx, int32_t e_lo, int32_t e_hi, int32_t m, const double *h_q, int64_t n) {
    if (!ctx) return NYXRT_EINVAL;
    CU(cudaSetDevice(ctx->g.device));
    if (!h_q) {                                                            // back to monochromatic: both tables go
        if (ctx->d_lut_t) cudaFree(ctx->d_lut_t);
        ctx->d_lut_t = nullptr;
        if (ctx->d_lut) cudaFree(ctx->d_lut);
        ctx->d_lut = nullptr;
        return NYXRT_OK;
    }
    // a rejected call changes nothing: both tables stay as they were until the new Q table is on the device
    int64_t need = 0;
    if (nyxrt_spectrum_nodes(e_lo, e_hi, m, &need) != NYXRT_OK || n != need)
        return fail(ctx, NYXRT_EINVAL, "set_spectrum: bad table geometry or length");
    if (geom_template(ctx->p.geom_mode) != 3)
        return fail(ctx, NYXRT_EINVAL, "set_spectrum: the spectrum table needs geom_mode 2 or 3");
    for (int64_t k = 0; k < n; ++k)
        if (!(h_q[k] >= 0.0) || !(h_q[k] <= 1.0) || (k > 0 && h_q[k] < h_q[k - 1]))
            return fail(ctx, NYXRT_EINVAL, "set_spectrum: Q must be non-decreasing within [0, 1]");
    double *d = nullptr;
    CU(cudaMalloc(&d, n * sizeof(double)));
    const cudaError_t ce = cudaMemcpy(d, h_q, n * sizeof(double), cudaMemcpyHostToDevice);
    if (ce != cudaSuccess) {
        cudaFree(d);
        return fail(ctx, NYXRT_ECUDA, "set_spectrum: copy failed: %s", cudaGetErrorString(ce));
    }
    if (ctx->d_lut_t) cudaFree(ctx->d_lut_t);                              // a new Q table drops the thin table
    ctx->d_lut_t = nullptr;
    if (ctx->d_lut) cudaFree(ctx->d_lut);
    ctx->d_lut = d;
    ctx->lut_e_lo = e_lo; ctx->lut_e_hi = e_hi; ctx->lut_m = m; ctx->lut_n = n;
    ctx->lut_first = h_q[0];
    ctx->lut_last = h_q[n - 1];
    return NYXRT_OK;
}

int nyxrt_set_spectrum_thin(nyxrt_ctx *ctx, const double *h_t, int64_t n, double tau_thin) {
    if (!ctx) return NYXRT_EINVAL;
    CU(cudaSetDevice(ctx->g.device));
    if (!h_t) {                                                            // thin table off
        if (ctx->d_lut_t) cudaFree(ctx->d_lut_t);
        ctx->d_lut_t = nullptr;
        return NYXRT_OK;
    }
    // as in set_spectrum: a rejected call leaves the thin table that was set before in place
    if (!ctx->d_lut) return fail(ctx, NYXRT_ESTATE, "set_spectrum_thin: set the Q table first");
    if (n != ctx->lut_n || !(tau_thin >= 0.0)) return fail(ctx, NYXRT_EINVAL, "set_spectrum_thin: bad length or threshold");
    for (int64_t k = 0; k < n; ++k)
        if (!(h_t[k] >= 0.0) || !(h_t[k] <= 1.0e300)) return fail(ctx, NYXRT_EINVAL, "set_spectrum_thin: T must be finite and >= 0");
    double *d = nullptr;
    CU(cudaMalloc(&d, n * sizeof(double)));
    const cudaError_t ce = cudaMemcpy(d, h_t, n * sizeof(double), cudaMemcpyHostToDevice);
    if (ce != cudaSuccess) {
        cudaFree(d);
        return fail(ctx, NYXRT_ECUDA, "set_spectrum_thin: copy failed: %s", cudaGetErrorString(ce));
    }
    if (ctx->d_lut_t) cudaFree(ctx->d_lut_t);
    ctx->d_lut_t = d;
    ctx->lut_t_first = h_t[0];
    ctx->lut_t_last = h_t[n - 1];
    ctx->tau_thin = tau_thin;
    return NYXRT_OK;
}

int nyxrt_blackbody_thin_table(double t_eff_K, int32_t e_lo, int32_t e_hi, int32_t m, double *h_t, int64_t n) {
    int64_t need = 0;
    if (!h_t || !(t_eff_K > 0.0) || nyxrt_spectrum_nodes(e_lo, e_hi, m, &need) != NYXRT_OK || n != need) return NYXRT_EINVAL;
    const double x0 = 13.598434 * 1.602176634e-19 / (1.380649e-23 * t_eff_K);   // h nu_0 / k T_eff
    const double norm = bb_absorbed(x0, 0.0, 0);
    for (int64_t k = 0; k < n; ++k) {
        double tau = 0.0;
        nyxrt_spectrum_node_tau(e_lo, m, k, &tau);
        h_t[k] = bb_absorbed(x0, tau, 2) / norm;
    }
    return NYXRT_OK;
}

int nyxrt_blackbody_table(double t_eff_K, int32_t e_lo, int32_t e_hi, int32_t m, double *h_q, int64_t n) {
    int64_t need = 0;
    if (!h_q || !(t_eff_K > 0.0) || nyxrt_spectrum_nodes(e_lo, e_hi, m, &need) != NYXRT_OK || n != need) return NYXRT_EINVAL;
    const double x0 = 13.598434 * 1.602176634e-19 / (1.380649e-23 * t_eff_K);   // h nu_0 / k T_eff
    const double norm = bb_absorbed(x0, 0.0, 0);
    for (int64_t k = 0; k < n; ++k) {
        double tau = 0.0;
        nyxrt_spectrum_node_tau(e_lo, m, k, &tau);
        const double q = bb_absorbed(x0, tau, 1) / norm;
        h_q[k] = q > 1.0 ? 1.0 : q;
        if (k > 0 && h_q[k] < h_q[k - 1]) h_q[k] = h_q[k - 1];              // quadrature noise near Q = 1
    }
    return NYXRT_OK;
}

int nyxrt_set_shard(nyxrt_ctx *ctx, int32_t rank, int32_t world) {
    if (!ctx) return NYXRT_EINVAL;
    if (world < 1 || rank < 0 || rank >= world) return fail(ctx, NYXRT_EINVAL, "set_shard: need 0 <= rank < world");
    ctx->shard_rank = rank;
    ctx->shard_world = world;
    return NYXRT_OK;
}

int nyxrt_trace_photons(nyxrt_ctx *ctx, double *d_photons, nyxrt_stats *hs, void *cuda_stream) {
    if (!ctx) return NYXRT_EINVAL;
    if (!d_photons) return fail(ctx, NYXRT_EINVAL, "trace_photons: null output");
    return run_trace(ctx, nullptr, nullptr, d_photons, hs, cuda_stream);
}

int nyxrt_finalise(nyxrt_ctx *ctx, const double *d_photons, double *d_gamma, double *d_heat, double *h_absorbed,
                   void *cuda_stream) {
    if (!ctx) return NYXRT_EINVAL;
    if (!d_photons || !d_gamma) return fail(ctx, NYXRT_EINVAL, "finalise: null pointer");
    if (!ctx->ws || !ctx->have_fields) return fail(ctx, NYXRT_ESTATE, "finalise: workspace and fields must be set first");
    cudaStream_t st = (cudaStream_t)cuda_stream;
    CU(cudaSetDevice(ctx->g.device));
    const double V = ctx->g.dx_cm * ctx->g.dx_cm * ctx->g.dx_cm;
    finalise_dense_kernel<<<NPARTIAL, 256, 0, st>>>(d_gamma, d_heat, d_photons, ctx->absorber, ctx->g.nx, ctx->g.ny,
                                                    ctx->g.nz, V, ctx->p.e_excess_erg, ctx->partial);
    sum_partials_kernel<<<1, 256, 0, st>>>(ctx->partial, NPARTIAL, ctx->scalars + 1);
    CU(cudaMemcpyAsync(ctx->h_scalars + 1, ctx->scalars + 1, sizeof(double), cudaMemcpyDeviceToHost, st));
    CU(cudaStreamSynchronize(st));
    CU(cudaGetLastError());
    if (h_absorbed) *h_absorbed = ctx->h_scalars[1];
    return NYXRT_OK;
}

int nyxrt_get_catalog(nyxrt_ctx *ctx, int64_t cap, int32_t *cell_ijk, double *L, double *radius, int64_t *n_out) {
    if (!ctx) return NYXRT_EINVAL;
    if (!n_out || cap < 0) return fail(ctx, NYXRT_EINVAL, "get_catalog: bad argument");
    if (!ctx->have_catalog) return fail(ctx, NYXRT_ESTATE, "get_catalog: no trace has run");
    CU(cudaSetDevice(ctx->g.device));
    *n_out = ctx->n_cat;
    const long long m = cap < ctx->n_cat ? cap : ctx->n_cat;
    if (m == 0) return NYXRT_OK;
    const SrcBufs &s = ctx->sb;
    if (cell_ijk) {
        int4 *tmp = new (std::nothrow) int4[m];
        if (!tmp) return fail(ctx, NYXRT_ENOMEM, "get_catalog: host allocation failed");
        cudaError_t e = cudaMemcpy(tmp, s.cell[0], m * sizeof(int4), cudaMemcpyDeviceToHost);
        for (long long a = 0; a < m && e == cudaSuccess; ++a) {
            cell_ijk[3 * a] = tmp[a].x; cell_ijk[3 * a + 1] = tmp[a].y; cell_ijk[3 * a + 2] = tmp[a].z;
        }
        delete[] tmp;
        CU(e);
    }
    if (L) CU(cudaMemcpy(L, s.L2[0], m * sizeof(double), cudaMemcpyDeviceToHost));
    if (radius) CU(cudaMemcpy(radius, s.r[0], m * sizeof(double), cudaMemcpyDeviceToHost));
    return NYXRT_OK;
}

int nyxrt_step_host(nyxrt_ctx *ctx, const void *h_nH, const void *h_xHI, int64_t n_src, const double *pos,
                    const double *L, double *h_gamma, double *h_heat, nyxrt_stats *hs) {
    if (!ctx) return NYXRT_EINVAL;
    if (!h_nH || !h_xHI || !h_gamma) return fail(ctx, NYXRT_EINVAL, "step_host: null pointer");
    if (!ctx->ws || !ctx->host_staging) return fail(ctx, NYXRT_ESTATE, "step_host: workspace lacks host staging");
    cudaStream_t st = ctx->own_stream;
    CU(cudaSetDevice(ctx->g.device));
    const size_t fb = (size_t)ctx->ncell * field_elem(ctx);
    CU(cudaMemcpyAsync(ctx->st_nH, h_nH, fb, cudaMemcpyHostToDevice, st));
    CU(cudaMemcpyAsync(ctx->st_xHI, h_xHI, fb, cudaMemcpyHostToDevice, st));
    int rc = nyxrt_set_fields(ctx, ctx->st_nH, ctx->st_xHI, st);
    if (rc) return rc;
    rc = nyxrt_set_sources(ctx, n_src, pos, L, st);
    if (rc) return rc;
    rc = nyxrt_trace(ctx, ctx->st_gamma, h_heat ? ctx->st_heat : nullptr, hs, st);
    if (rc) return rc;
    CU(cudaMemcpyAsync(h_gamma, ctx->st_gamma, ctx->ncell * sizeof(double), cudaMemcpyDeviceToHost, st));
    if (h_heat) CU(cudaMemcpyAsync(h_heat, ctx->st_heat, ctx->ncell * sizeof(double), cudaMemcpyDeviceToHost, st));
    CU(cudaStreamSynchronize(st));
    return NYXRT_OK;
}

int nyxrt_timestep(nyxrt_ctx *ctx, const nyxrt_ode *ode, const void *d_nH, const double *d_y_begin, double *d_y_end,
                   void *d_y_avg, double *d_gamma, double *d_heat, nyxrt_stats *hs, nyxrt_tstats *ht, void *cuda_stream) {
    if (!ctx) return NYXRT_EINVAL;
    if (!ode || !d_nH || !d_y_begin || !d_y_end || !d_y_avg || !d_gamma)
        return fail(ctx, NYXRT_EINVAL, "timestep: null pointer");
    const nyxrt_ode &o = *ode;
    if (!(o.dt_s > 0.0) || o.max_iter < 1 || o.inner_iter < 1 || !(o.alpha_cm3_s >= 0.0) || !(o.coll_cm3_s >= 0.0) ||
        !(o.clumping >= 0.0) || !(o.tol_rel >= 0.0) || !(o.tol_abs >= 0.0) || !(o.unconv_frac >= 0.0))
        return fail(ctx, NYXRT_EINVAL, "timestep: bad parameters");
    if (!ctx->ws || !ctx->have_sources) return fail(ctx, NYXRT_ESTATE, "timestep: workspace and sources must be set first");
    cudaStream_t st = (cudaStream_t)cuda_stream;
    CU(cudaSetDevice(ctx->g.device));
    const long long n = ctx->ncell;
    const bool f32 = ctx->g.field_dtype != 0;
    const OdeArgs oa{o.dt_s, o.alpha_cm3_s, o.coll_cm3_s, o.clumping, o.tol_rel, o.tol_abs, o.inner_iter};
    unsigned long long *conv = reinterpret_cast<unsigned long long *>(ctx->scalars + 4);
    nyxrt_tstats t;
    memset(&t, 0, sizeof t);
    nyxrt_stats s_last;
    memset(&s_last, 0, sizeof s_last);
    cudaEvent_t e0 = ctx->tev[0], e1 = ctx->tev[1], e2 = ctx->tev[2], e3 = ctx->tev[3];
    CU(cudaEventRecord(e0, st));
    if (f32) init_avg_kernel<float><<<NPARTIAL, 256, 0, st>>>(d_y_begin, (float *)d_y_avg, n);
    else init_avg_kernel<double><<<NPARTIAL, 256, 0, st>>>(d_y_begin, (double *)d_y_avg, n);
    t.kernel_launches = 1;
    double ms_rt = 0.0, ms_ode = 0.0;
    for (int it = 0; it < o.max_iter; ++it) {
        int rc = nyxrt_set_fields(ctx, d_nH, d_y_avg, st);
        if (rc) return rc;
        rc = nyxrt_trace(ctx, d_gamma, d_heat, &s_last, st);
        if (rc) return rc;
        t.iterations = it + 1;
        t.segments_total += s_last.segments;
        t.kernel_launches += s_last.kernel_launches + 2 + 1;          // + prep_fields, sum_partials, ode
        ms_rt += s_last.ms_total;
        CU(cudaEventRecord(e1, st));
        CU(cudaMemsetAsync(conv, 0, 2 * sizeof(unsigned long long), st));
        if (f32) ode_kernel<float><<<NPARTIAL, 256, 0, st>>>(d_gamma, (const float *)d_nH, d_y_begin, (float *)d_y_avg, d_y_end, n, oa, conv);
        else ode_kernel<double><<<NPARTIAL, 256, 0, st>>>(d_gamma, (const double *)d_nH, d_y_begin, (double *)d_y_avg, d_y_end, n, oa, conv);
        CU(cudaEventRecord(e2, st));
        CU(cudaMemcpyAsync(ctx->h_scalars + 4, conv, 2 * sizeof(unsigned long long), cudaMemcpyDeviceToHost, st));
        CU(cudaStreamSynchronize(st));
        CU(cudaGetLastError());
        float ms = 0.f;
        cudaEventElapsedTime(&ms, e1, e2);
        ms_ode += ms;
        unsigned long long hv[2];
        memcpy(hv, ctx->h_scalars + 4, sizeof hv);
        t.unconverged_cells = hv[0];
        memcpy(&t.max_rel_change, &hv[1], sizeof(double));
        if ((double)hv[0] <= o.unconv_frac * (double)n) { t.converged = 1; break; }
    }
    CU(cudaEventRecord(e3, st));
    CU(cudaEventSynchronize(e3));
    cudaEventElapsedTime(&t.ms_total, e0, e3);
    t.ms_rt = (float)ms_rt;
    t.ms_ode = (float)ms_ode;
    if (hs) *hs = s_last;
    if (ht) *ht = t;
    return NYXRT_OK;
}

int nyxrt_pix2dir(nyxrt_ctx *ctx, int32_t level, int64_t pix_begin, int64_t n, double *dir_xyz) {
    if (!ctx) return NYXRT_EINVAL;
    if (level < 0 || level > 14 || pix_begin < 0 || n < 0 || !dir_xyz || pix_begin + n > (12ll << (2 * level)))
        return fail(ctx, NYXRT_EINVAL, "pix2dir: bad argument");
    if (n == 0) return NYXRT_OK;
    CU(cudaSetDevice(ctx->g.device));
    double *d = nullptr;
    CU(cudaMalloc(&d, 3 * n * sizeof(double)));
    pix2dir_kernel<<<blocks_for(n, 128), 128>>>(level, pix_begin, n, d);
    cudaError_t e = cudaMemcpy(dir_xyz, d, 3 * n * sizeof(double), cudaMemcpyDeviceToHost);
    cudaFree(d);
    CU(e);
    return NYXRT_OK;
}

}  // extern "C"
