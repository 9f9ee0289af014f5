// bte_pendulum.cuh -- zero-temperature limit of the model, eq. (44)-(46).
//
// One electron starts at (phi_x, phi_y) = (0, 0) at time t0 and follows d phi_x/dt = E(t) + B phi_y (44),
// d phi_y/dt = -B sin(phi_x) (45); its velocity sin(phi_x) enters the drift velocity through the exponential memory
// (46).  Averaged over one ac period:  <v_dr g(t)> = (1/T) int_0^T dt0 int_0^inf ds e^{-s} sin phi_x(t0+s; t0) g(t0+s),
// g = 1, cos wt, sin wt.  Discretisation (C20): classical RK4 with step h, composite Simpson on the RK4 nodes
// (memory cut at n_rk h), rectangle rule over n_phase start phases.  Plain fp64 ALU work, embarrassingly parallel:
// one CTA per parameter set, one thread per start phase (strided), deterministic block reduction.
#pragma once
#include <cuda_runtime.h>

namespace bte {

struct PendulumParams { double E_dc, E_omega, omega, B; };
struct PendulumOut { double v_mean, v_cos, v_sin; };

__device__ __forceinline__ void pendulum_rhs(const PendulumParams& p, double t, double px, double py, double& dx,
                                             double& dy) {
    dx = (p.E_dc + p.E_omega * cos(p.omega * t)) + p.B * py;
    dy = -p.B * sin(px);
}

__global__ void __launch_bounds__(128) pendulum_kernel(const PendulumParams* __restrict__ params,
                                                       PendulumOut* __restrict__ out, int n_phase, double h,
                                                       int n_rk) {
    __shared__ double red[3][128];
    const PendulumParams p = params[blockIdx.x];
    const bool ac = (p.E_omega != 0.0) && (p.omega != 0.0);
    const int P = ac ? n_phase : 1;
    const double T = ac ? 2.0 * 3.14159265358979323846 / p.omega : 0.0;
    double sum0 = 0.0, sumc = 0.0, sums = 0.0;
    for (int j = threadIdx.x; j < P; j += blockDim.x) {
        const double t0 = ac ? T * j / P : 0.0;
        double px = 0.0, py = 0.0, I0 = 0.0, Ic = 0.0, Is = 0.0;
        for (int k = 0; k <= n_rk; ++k) {
            const double s = k * h, t = t0 + s;
            const double wgt = (k == 0 || k == n_rk) ? 1.0 : ((k & 1) ? 4.0 : 2.0);
            const double g = exp(-s) * sin(px);
            double sn, cs;
            sincos(p.omega * t, &sn, &cs);
            I0 += wgt * g;
            Ic += wgt * g * cs;
            Is += wgt * g * sn;
            if (k == n_rk) break;
            double k1x, k1y, k2x, k2y, k3x, k3y, k4x, k4y;
            pendulum_rhs(p, t, px, py, k1x, k1y);
            pendulum_rhs(p, t + 0.5 * h, px + 0.5 * h * k1x, py + 0.5 * h * k1y, k2x, k2y);
            pendulum_rhs(p, t + 0.5 * h, px + 0.5 * h * k2x, py + 0.5 * h * k2y, k3x, k3y);
            pendulum_rhs(p, t + h, px + h * k3x, py + h * k3y, k4x, k4y);
            px += (h / 6.0) * (k1x + 2.0 * k2x + 2.0 * k3x + k4x);
            py += (h / 6.0) * (k1y + 2.0 * k2y + 2.0 * k3y + k4y);
        }
        sum0 += I0 * (h / 3.0);
        sumc += Ic * (h / 3.0);
        sums += Is * (h / 3.0);
    }
    red[0][threadIdx.x] = sum0; red[1][threadIdx.x] = sumc; red[2][threadIdx.x] = sums;
    __syncthreads();
    for (int o = 64; o > 0; o >>= 1) {                      // fixed tree => deterministic
        if (threadIdx.x < o) {
#pragma unroll
            for (int q = 0; q < 3; ++q) red[q][threadIdx.x] += red[q][threadIdx.x + o];
        }
        __syncthreads();
    }
    if (threadIdx.x == 0) {
        out[blockIdx.x].v_mean = red[0][0] / P;
        out[blockIdx.x].v_cos = red[1][0] / P;
        out[blockIdx.x].v_sin = red[2][0] / P;
    }
}

}  // namespace bte
