/* A plain C client of include/nyxrt.h (no Python, no torch): config 1 of BASELINE.json -- the 32^3 Stroemgren
 * test -- through the C ABI with cudaMalloc'ed buffers.  Built and run by tests/test_gpu_cabi.py, which compares
 * the numbers printed here with the Python binding's and the oracle's.  Prints one line:
 *   segments spawned0..4 killed_tau_total photons_absorbed photons_emitted sum_gamma gamma_at_source_neighbour */
#include <cuda_runtime.h>
#include <stdio.h>
#include <stdlib.h>
#include <string.h>

#include "nyxrt.h"

#define CHECK(call) do { int rc_ = (call); if (rc_ != NYXRT_OK) { \
    fprintf(stderr, "%s -> %d: %s\n", #call, rc_, ctx ? nyxrt_last_error(ctx) : ""); return 2; } } while (0)

int main(void) {
    const int n = 32;
    const size_t ncell = (size_t)n * n * n;
    nyxrt_ctx *ctx = NULL;
    nyxrt_grid g;
    nyxrt_params p;
    memset(&g, 0, sizeof g);
    memset(&p, 0, sizeof p);
    g.nx = g.ny = g.nz = n;
    g.field_dtype = 0;
    g.dx_cm = 6.6 * 3.0856775814913673e21 / n;       /* box 6.6 kpc */
    g.pos_unit_cm = g.dx_cm;                         /* source positions in cells */
    p.sigma_cm2 = 6.3e-18; p.n_min_ray = 3.0; p.tau_max = 18.420680743952367; /* ln 1e8 */
    p.automerge_xmean = 0.018; p.delta_r = 2.0; p.r_max = 8.0; p.f_ov = 1.0; p.x_th = 0.9; p.f_req = 0.75; p.eps = 1e-9;
    p.level_max = 13; p.geom_mode = 3; p.merge = 0; p.n_min_samples = 16; p.samp_level = 2;
    if (nyxrt_sizeof_grid() != (int)sizeof g || nyxrt_sizeof_params() != (int)sizeof p ||
        nyxrt_sizeof_stats() != (int)sizeof(nyxrt_stats)) { fprintf(stderr, "struct size mismatch\n"); return 3; }
    CHECK(nyxrt_create(&g, &p, &ctx));
    uint64_t ws_bytes = 0;
    CHECK(nyxrt_workspace_bytes(ctx, 1, 0, 0, &ws_bytes));
    void *ws = NULL;
    double *d_nH = NULL, *d_xHI = NULL, *d_gamma = NULL, *d_heat = NULL;
    if (cudaMalloc(&ws, ws_bytes) || cudaMalloc((void **)&d_nH, ncell * 8) || cudaMalloc((void **)&d_xHI, ncell * 8) ||
        cudaMalloc((void **)&d_gamma, ncell * 8) || cudaMalloc((void **)&d_heat, ncell * 8)) return 4;
    double *h = (double *)malloc(ncell * 8);
    for (size_t i = 0; i < ncell; ++i) h[i] = 1e-3;
    cudaMemcpy(d_nH, h, ncell * 8, cudaMemcpyHostToDevice);
    for (size_t i = 0; i < ncell; ++i) h[i] = 1.0;
    cudaMemcpy(d_xHI, h, ncell * 8, cudaMemcpyHostToDevice);
    CHECK(nyxrt_set_workspace(ctx, ws, ws_bytes, 1, 0, 0));
    CHECK(nyxrt_set_fields(ctx, d_nH, d_xHI, NULL));
    const double pos[3] = {16.5, 16.5, 16.5}, L[1] = {5e48};
    CHECK(nyxrt_set_sources(ctx, 1, pos, L, NULL));
    nyxrt_stats st;
    CHECK(nyxrt_trace(ctx, d_gamma, d_heat, &st, NULL));
    cudaMemcpy(h, d_gamma, ncell * 8, cudaMemcpyDeviceToHost);
    double sum = 0.0;
    for (size_t i = 0; i < ncell; ++i) sum += h[i];
    uint64_t kt = 0;
    for (int l = 0; l < NYXRT_MAXLEV; ++l) kt += st.killed_tau[l];
    printf("%llu %llu %llu %llu %llu %llu %llu %.17g %.17g %.17g %.17g\n", (unsigned long long)st.segments,
           (unsigned long long)st.spawned[0], (unsigned long long)st.spawned[1], (unsigned long long)st.spawned[2],
           (unsigned long long)st.spawned[3], (unsigned long long)st.spawned[4], (unsigned long long)kt,
           st.photons_absorbed, st.photons_emitted, sum, h[((size_t)16 * n + 16) * n + 17]);
    int32_t cell[3]; double cl, cr; int64_t ncat = 0;
    CHECK(nyxrt_get_catalog(ctx, 1, cell, &cl, &cr, &ncat));
    if (ncat != 1 || cell[0] != 16 || cell[1] != 16 || cell[2] != 16 || cl != 5e48) return 5;
    /* error path: tracing after the sources were dropped by a bad call */
    const double bad[3] = {40.0, 1.0, 1.0};
    if (nyxrt_set_sources(ctx, 1, bad, L, NULL) != NYXRT_EINVAL) return 6;
    if (nyxrt_trace(ctx, d_gamma, NULL, NULL, NULL) != NYXRT_ESTATE) return 7;
    nyxrt_destroy(ctx);
    cudaFree(ws); cudaFree(d_nH); cudaFree(d_xHI); cudaFree(d_gamma); cudaFree(d_heat);
    free(h);
    return 0;
}
