// finalise_static.cu -- nyxrt_finalise_static: the last stage of the RT step (row a9: Gamma = photons / (n_HI V),
// Eq. 1 with V_box; heating, reading H1) for a caller that must not allocate device memory.
//
// Who that is.  This library normally lives inside someone else's memory manager: Nyx runs on AMReX, whose arena
// takes almost all of the GPU's memory when the code starts, and the Python binding here runs under PyTorch's
// caching allocator, which does the same over time.  In both, a plain cudaMalloc issued by a plug-in can fail
// although the host code still has plenty of free blocks, and cudaMalloc / cudaFree make the whole device wait,
// which stalls the hydro or training streams running next to the RT step.  The other entry points avoid this with
// a context (nyxrt_create: a few small allocations, once) and a caller-provided workspace.  A caller that cannot
// afford even that -- a post-processing rank of a source-sharded job that only receives the all-reduced photon
// grid, a one-off diagnostic inside a time step -- gets this one call: no context, no workspace, nothing allocated.
//
// The scratch of the reduction (one partial sum per grid row) therefore sits in a file-scope device array of fixed
// size, NYXRT_STATIC_MAX_ROWS doubles = 8 MiB, which every GPU that loads libnyxrt.so holds until the process ends.
// Consequences, also stated in include/nyxrt.h:
//   - grids with more than NYXRT_STATIC_MAX_ROWS rows (ny * nz) are refused, never truncated;
//   - the array is shared by all calls in the process and keeps what the last call left in it.  Nothing in it has
//     to start at zero: the second kernel reads exactly the ny * nz partials the first kernel of the same call has
//     just overwritten, and nothing beyond them;
//   - two calls whose kernels overlap on one GPU (different streams, or different host threads) race on it.
//     Calls on one stream, or calls ordered by events, are safe;
//   - the array's name in host code is only a handle: the device address is asked for once per device with
//     cudaGetSymbolAddress, on the first call that names that device.  That first call should be made outside any
//     stream capture.
#include <cuda_runtime.h>

#include <cstdarg>
#include <cstdio>
#include <mutex>

#include "../../include/nyxrt.h"

namespace {

constexpr int MAX_DEVICES = 64;
constexpr int ROW_WARPS = 8;                       // warps (= rows in flight) per block of the row kernel
constexpr int SUM_THREADS = 1024;

// One partial sum per grid row (fixed j, k).  Device code below names it directly; host code must not pass this
// name to a kernel (see set-up in nyxrt_finalise_static).
static __device__ __align__(256) double g_row_partial[NYXRT_STATIC_MAX_ROWS];

std::mutex g_setup_mutex;
double *g_scratch_of_device[MAX_DEVICES];          // device address of g_row_partial, per device ordinal (NULL: not asked yet)

// The variant of finalise_dense_kernel (march.cuh): same per-cell arithmetic -- ph / (|n_H x_HI| V) and
// (e_excess ph) / V, exactly 0 where no photon arrived -- with the absorber density formed from the caller's fields
// instead of the context's padded copy (the product n_H x_HI in fp64 is what set_fields stores, up to the sign bit
// that fabs removes).  One warp per row, lanes along x (coalesced); the row's photons are summed per lane in x
// order and then across lanes by a fixed butterfly, so the partial of a row depends on nx alone.
template <typename T>
__global__ void finalise_rows_kernel(double *__restrict__ gamma, double *__restrict__ heat,
                                     const double *__restrict__ photons, const T *__restrict__ nH,
                                     const T *__restrict__ xHI, int nx, long long nrow, double V, double e_excess,
                                     double *__restrict__ row_partial) {
    const int lane = threadIdx.x & 31;
    const long long warp = (long long)blockIdx.x * ROW_WARPS + (threadIdx.x >> 5);
    const long long nwarp = (long long)gridDim.x * ROW_WARPS;
    for (long long row = warp; row < nrow; row += nwarp) {
        const long long base = row * nx;
        double sum = 0.0;
        for (int i = lane; i < nx; i += 32) {
            const long long t = base + i;
            const double ph = photons[t];
            sum += ph;
            double g = 0.0, h = 0.0;
            if (ph != 0.0) {
                const double a = (double)nH[t] * (double)xHI[t];
                g = ph / (fabs(a) * V);
                h = e_excess * ph / V;
            }
            gamma[t] = g;
            if (heat) heat[t] = h;
        }
        for (int o = 16; o > 0; o >>= 1) sum += __shfl_xor_sync(0xffffffffu, sum, o);
        if (lane == 0) row_partial[row] = sum;
    }
}

// Fixed-order sum of the first nrow partials: thread t adds rows t, t + 1024, ... in that order, then a tree.
__global__ void sum_rows_kernel(const double *__restrict__ row_partial, long long nrow, double *__restrict__ out) {
    __shared__ double sh[SUM_THREADS];
    double acc = 0.0;
    for (long long r = threadIdx.x; r < nrow; r += SUM_THREADS) acc += row_partial[r];
    sh[threadIdx.x] = acc;
    __syncthreads();
    for (int o = SUM_THREADS >> 1; o > 0; o >>= 1) {
        if ((int)threadIdx.x < o) sh[threadIdx.x] += sh[threadIdx.x + o];
        __syncthreads();
    }
    if (threadIdx.x == 0) *out = sh[0];
}

int refuse(char *errbuf, int64_t errbuf_len, int code, const char *fmt, ...) {
    if (errbuf && errbuf_len > 0) {
        va_list ap;
        va_start(ap, fmt);
        vsnprintf(errbuf, (size_t)errbuf_len, fmt, ap);
        va_end(ap);
    }
    return code;
}

}  // namespace

extern "C" int nyxrt_finalise_static(int32_t device, int32_t nx, int32_t ny, int32_t nz, int32_t field_dtype,
                                     double dx_cm, double e_excess_erg, const void *d_nH, const void *d_xHI,
                                     const double *d_photons, double *d_gamma_HI, double *d_heat,
                                     double *d_absorbed, void *cuda_stream, char *errbuf, int64_t errbuf_len) {
    if (errbuf && errbuf_len > 0) errbuf[0] = 0;
    if (device < 0 || device >= MAX_DEVICES)
        return refuse(errbuf, errbuf_len, NYXRT_EINVAL, "finalise_static: device ordinal %d outside 0..%d", device, MAX_DEVICES - 1);
    if (nx < 1 || ny < 1 || nz < 1 || nx > (1 << 20) || ny > (1 << 20) || nz > (1 << 20))
        return refuse(errbuf, errbuf_len, NYXRT_EINVAL, "finalise_static: each of nx, ny, nz must be 1..2^20");
    if (field_dtype != 0 && field_dtype != 1)
        return refuse(errbuf, errbuf_len, NYXRT_EINVAL, "finalise_static: field_dtype must be 0 (fp64) or 1 (fp32)");
    if (!(dx_cm > 0.0) || !(e_excess_erg >= 0.0))
        return refuse(errbuf, errbuf_len, NYXRT_EINVAL, "finalise_static: need dx_cm > 0 and e_excess_erg >= 0");
    if (!d_nH || !d_xHI || !d_photons || !d_gamma_HI)
        return refuse(errbuf, errbuf_len, NYXRT_EINVAL, "finalise_static: null pointer (only d_heat and d_absorbed may be NULL)");
    const long long nrow = (long long)ny * nz;
    if (nrow > (long long)NYXRT_STATIC_MAX_ROWS)
        return refuse(errbuf, errbuf_len, NYXRT_ENOMEM,
                      "finalise_static: ny * nz = %lld rows, the fixed scratch holds %d (NYXRT_STATIC_MAX_ROWS); "
                      "use nyxrt_finalise with a context and workspace for larger grids", nrow, (int)NYXRT_STATIC_MAX_ROWS);

    cudaError_t e = cudaSetDevice(device);
    if (e != cudaSuccess)
        return refuse(errbuf, errbuf_len, NYXRT_ECUDA, "finalise_static: cudaSetDevice(%d): %s", device, cudaGetErrorString(e));
    // Set-up, once per device, with that device current: the device address behind the symbol.
    double *scratch = nullptr;
    {
        std::lock_guard<std::mutex> lock(g_setup_mutex);
        if (!g_scratch_of_device[device]) {
            void *p = nullptr;
            e = cudaGetSymbolAddress(&p, g_row_partial);
            if (e != cudaSuccess || !p)
                return refuse(errbuf, errbuf_len, NYXRT_ECUDA, "finalise_static: cudaGetSymbolAddress on device %d: %s", device,
                              cudaGetErrorString(e));
            g_scratch_of_device[device] = static_cast<double *>(p);
        }
        scratch = g_scratch_of_device[device];
    }

    cudaStream_t st = (cudaStream_t)cuda_stream;
    const double V = dx_cm * dx_cm * dx_cm;
    const long long want = (nrow + ROW_WARPS - 1) / ROW_WARPS;
    const int blocks = (int)(want < 148 * 8 ? want : 148 * 8);             // 8 blocks of 256 threads per SM, rows strided
    if (field_dtype)
        finalise_rows_kernel<float><<<blocks, 32 * ROW_WARPS, 0, st>>>(d_gamma_HI, d_heat, d_photons, (const float *)d_nH,
                                                                     (const float *)d_xHI, nx, nrow, V, e_excess_erg, scratch);
    else
        finalise_rows_kernel<double><<<blocks, 32 * ROW_WARPS, 0, st>>>(d_gamma_HI, d_heat, d_photons, (const double *)d_nH,
                                                                      (const double *)d_xHI, nx, nrow, V, e_excess_erg, scratch);
    if (d_absorbed) sum_rows_kernel<<<1, SUM_THREADS, 0, st>>>(scratch, nrow, d_absorbed);
    e = cudaGetLastError();
    if (e != cudaSuccess)
        return refuse(errbuf, errbuf_len, NYXRT_ECUDA, "finalise_static: launch failed: %s", cudaGetErrorString(e));
    return NYXRT_OK;
}
