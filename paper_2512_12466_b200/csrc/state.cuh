// Device-resident state shared by the kernels of one context.
#pragma once
#include <stdint.h>

namespace nyxrt {

constexpr int MAXLEV = 16;

// Ray key: [src:30][level:4][pix:30].  pix < 12*4^13 < 2^30.
__host__ __device__ __forceinline__ uint64_t ray_key(uint32_t src, int level, uint32_t pix) {
    return ((uint64_t)src << 34) | ((uint64_t)level << 30) | (uint64_t)pix;
}
__host__ __device__ __forceinline__ uint32_t key_src(uint64_t k) { return (uint32_t)(k >> 34); }
__host__ __device__ __forceinline__ uint32_t key_pix(uint64_t k) { return (uint32_t)(k & 0x3fffffffu); }

// The ray store: one SoA stack per HEALPix level inside one allocation (32 bytes per ray).
struct RayPool {
    uint64_t *key;
    double *s, *tau, *N;                 // distance travelled [cells], optical depth, photons/s carried
    long long off[MAXLEV];               // first slot of level l
    long long cap[MAXLEV];               // slots of level l
};

// Loop control, written by sched_kernel and read by emit/march (no host round trip per iteration).
struct LoopState {
    long long count[MAXLEV];             // rays on the stack of level l
    long long src_next, n_cat;           // catalogue cursor
    long long batch_rays;                // B
    long long begin, batch;              // march: slots [begin, begin+batch) of level `level` (popped)
    long long emit_src, emit_n, emit_slot;  // emit: sources [emit_src, emit_src+emit_n) -> level-0 slots
    int level;
    int done;
    int overflow;
    int seg_round;                       // cells marched per round, between two retire / pop passes
    unsigned long long iterations, peak_pool;
    unsigned long long fetch;            // next unclaimed ray of the current batch (chunks of FETCH_CHUNK)
};

struct DevStats {
    unsigned long long spawned[MAXLEV], split[MAXLEV], killed_tau[MAXLEV], exited[MAXLEV], killed_lmax[MAXLEV];
    unsigned long long holes[MAXLEV];   // filler slots popped at level l (slab padding; not rays)
    unsigned long long segments, zero_len, nbr_deposits;
    double escaped, residual, lost;
    double absorbed;                     // finalise: sum over cells
    double emitted;
};

constexpr uint64_t KEY_HOLE = ~0ull;     // filler slot (end of a warp's child slab)
constexpr int CHILD_SLAB = 128;          // child slots a warp reserves per atomic (>= 4 * 32)
constexpr int FETCH_CHUNK = 32;          // rays a warp claims per atomic (small: the end of a batch is shared evenly)

struct MarchArgs {
    const double *absorber;              // PADDED grid (nx+2)(ny+2)(nz+2): |a| = n_H x_HI; sign bit set where
                                         // n_H < n_th (Eq. 7-8 flag); halo = -inf (outside the box), or the
                                         // wrapped image of the opposite side in a periodic box
    double *acc;                         // PADDED: photons absorbed per cell
    const int4 *cat_cell;                // (i, j, k, 0) per catalogue source
    const double *cat_L;
    RayPool pool;
    LoopState *ls;
    DevStats *ds;
    int nx, ny, nz, level_max;
    long long px, pxy;                   // padded strides: px = nx+2, pxy = (nx+2)(ny+2)
    double sdx;                          // sigma * dx: optical depth per unit absorber per cell length
    double tau_max;
    double s_max;                        // periodic box: a ray ends once its travel distance s >= sqrt(nx^2+ny^2+nz^2)
                                         // cells = sqrt(3) L_box for a cube
    // spectrum table, used by the LUT instantiations only
    const double *lut_q;                 // Q at the nodes
    const double *lut_t;                 // T = dQ/dtau_0 at the nodes (thin segments), or null
    double lut_t_first, lut_t_last, tau_thin;
    double lut_t_lo, lut_t_hi, lut_inv_t_lo, lut_q_first, lut_q_last, lut_fscale;
    long long lut_k0, lut_fmask;
    int lut_fb;
    double r2_split[MAXLEV];             // Eq. 4: split when s^2 > 3 4^l / (pi N_min)
    double K[MAXLEV];                    // sqrt(Omega(l)) = sqrt(pi/3) 2^-l: L_pix = R K
};

}  // namespace nyxrt
