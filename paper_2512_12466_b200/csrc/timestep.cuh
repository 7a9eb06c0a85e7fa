// The RT timestep on the device (monochromatic): time integration of Eq. 3
// with the time-averaged semi-analytic solution of [23] (C2-Ray), used inside the
// iterative nonlinear solve of PAPER.md:105-107.  One thread per cell; the ray trace between two updates
// is the hot path of march.cuh.  Readings R32-R36.
#pragma once
#include <stdint.h>

namespace nyxrt {

struct OdeArgs {
    double dt, alpha, coll, clumping, tol_rel, tol_abs;
    int inner_iter;
};

// x_HI field of the first ray trace = the neutral fraction at the start of the step (R36)
template <typename T>
__global__ void init_avg_kernel(const double *__restrict__ y_begin, T *__restrict__ y_avg, long long n) {
    for (long long c = (long long)blockIdx.x * blockDim.x + threadIdx.x; c < n; c += (long long)gridDim.x * blockDim.x)
        y_avg[c] = (T)y_begin[c];
}

// Eq. 3 for the NEUTRAL fraction y = 1 - x with Gamma fixed:
//   dy/dt = a_rec - y (a_ion + a_rec),  a_ion = Gamma + n_e C_H,  a_rec = n_e alpha_H C,  n_e = <x> n_H (R33)
//   y(dt) = y_eq + (y0 - y_eq) e^{-w},  <y> = y_eq + (y0 - y_eq)(1 - e^{-w})/w,  w = (a_ion + a_rec) dt,
// <y> feeding n_e again inner_iter times (R34).  conv[0] counts the cells whose <y> moved by more than
// tol_rel <y> + tol_abs since the last iteration (R35), conv[1] holds the bits of the largest ratio
// (non-negative doubles order like their bit patterns).
template <typename T>
__global__ void ode_kernel(const double *__restrict__ gamma, const T *__restrict__ nH, const double *__restrict__ y_begin,
                           T *__restrict__ y_avg, double *__restrict__ y_end, long long n, OdeArgs o,
                           unsigned long long *conv) {
    unsigned long long bad = 0;
    double worst = 0.0;
    for (long long c = (long long)blockIdx.x * blockDim.x + threadIdx.x; c < n; c += (long long)gridDim.x * blockDim.x) {
        const double g = gamma[c], nh = (double)nH[c], y0 = y_begin[c], y_old = (double)y_avg[c];
        double yavg = y_old, yend = y0;
        for (int it = 0; it < o.inner_iter; ++it) {
            const double yprev = yavg;
            const double ne = (1.0 - yavg) * nh;
            const double a_ion = g + ne * o.coll;
            const double a_rec = (ne * o.alpha) * o.clumping;
            const double rate = a_ion + a_rec;
            const double w = rate * o.dt;
            if (!(w > 0.0)) { yend = y0; yavg = y0; break; }
            const double yeq = a_rec / rate;
            const double em1 = expm1(-w);
            yend = yeq + (y0 - yeq) * (1.0 + em1);
            yavg = yeq + (y0 - yeq) * (-em1 / w);
            yend = yend < 0.0 ? 0.0 : (yend > 1.0 ? 1.0 : yend);
            yavg = yavg < 0.0 ? 0.0 : (yavg > 1.0 ? 1.0 : yavg);
            if (yavg == yprev) break;        // a fixed point, bit for bit: the remaining iterations would repeat it
        }
        const T stored = (T)yavg;
        y_avg[c] = stored;
        y_end[c] = yend;
        const double y_new = (double)stored;
        const double lim = o.tol_rel * y_new + o.tol_abs;
        const double dy = fabs(y_new - y_old);
        if (dy > lim) ++bad;
        const double q = lim > 0.0 ? dy / lim : (dy > 0.0 ? CUDART_INF : 0.0);
        if (q > worst) worst = q;
    }
#pragma unroll
    for (int s = 16; s > 0; s >>= 1) {
        bad += __shfl_xor_sync(0xffffffffu, bad, s);
        const double w2 = __shfl_xor_sync(0xffffffffu, worst, s);
        worst = w2 > worst ? w2 : worst;
    }
    if ((threadIdx.x & 31) == 0) {
        if (bad) atomicAdd(conv, bad);
        if (worst > 0.0) atomicMax(conv + 1, (unsigned long long)__double_as_longlong(worst));
    }
}

}  // namespace nyxrt
