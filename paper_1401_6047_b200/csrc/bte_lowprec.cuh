// bte_lowprec.cuh -- fp32 variants of the step: the paper ran in float throughout
// and saw the norm of f drift for small time steps (L328).
//   PREC 1: the state is STORED as fp32 pairs (half the bytes per lattice point), arithmetic in fp64 (cn_point)
//   PREC 2: fp32 storage and fp32 arithmetic, operation by operation as the plain loop nest of the paper would do it
//           in float (explicit round-to-nearest intrinsics, no FMA contraction, IEEE division): bit-reproducible
//           against a CPU float implementation.
// Kernels: one thread per lattice point, two launches per step plus the reduction (the "split" form of the step;
// the streaming / resident kernels are fp64-only).  Reductions (reduce_finalize_kernel<float2>) accumulate in fp64.
#pragma once
#include "bte_kernels.cuh"

namespace bte {

__device__ __forceinline__ float2* state32_ptr(const Layout& L, int buf, int grid, int sys) {
    return (float2*)L.state + (((size_t)buf * 2 + grid) * L.n_batch + sys) * grid_points(L) + (size_t)GHOST * L.pitch;
}

__global__ void init_state32_kernel(Layout L, int prec) {
    const int sys = blockIdx.z, n = blockIdx.y;
    const int m = blockIdx.x * blockDim.x + threadIdx.x;
    if (blockIdx.x == 0 && n == 0 && threadIdx.x == 0) {
        SysState z = {};
        L.ss[sys] = z;
    }
    if (m >= L.pitch) return;
    float2 w = make_float2(0.f, 0.f);
    if (m < L.M1) {
        const double c = cn_ptr(L, sys)[n], g = L.gm[(size_t)sys * L.pitch + m];
        w.x = prec == 2 ? __fmul_rn((float)c, (float)g) : (float)(c * g);
    }
    state32_ptr(L, 0, 0, sys)[(size_t)n * L.pitch + m] = w;
}

// One application of T to one grid (modes as half_update_kernel: 0 whole, 1 fractional, 2 start-up).
template <int PREC>
__global__ void __launch_bounds__(128) half_update32_kernel(Layout L, int mode) {
    const int sys = blockIdx.z, n = blockIdx.y;
    const int m = blockIdx.x * blockDim.x + threadIdx.x;
    const SysConst c = L.sc[sys];
    const long long k = (mode == 2) ? 0 : L.ss[sys].k;
    if (mode != 2 && c.n_steps_total > 0 && k >= c.n_steps_total) return;   // frozen system
    const int cur = (mode == 2) ? 0 : L.ss[sys].buf, nxt = cur ^ 1;
    const float2 *X, *S;
    float2* O;
    double delta, ta, tb;
    if (mode == 0) {
        X = state32_ptr(L, cur, 0, sys); S = state32_ptr(L, cur, 1, sys); O = state32_ptr(L, nxt, 0, sys);
        delta = L.dt; ta = (double)k * L.dt; tb = ((double)k + 1.0) * L.dt;
    } else if (mode == 1) {
        X = state32_ptr(L, cur, 1, sys); S = state32_ptr(L, nxt, 0, sys); O = state32_ptr(L, nxt, 1, sys);
        delta = L.dt; ta = ((double)k + 0.5) * L.dt; tb = ((double)k + 1.5) * L.dt;
    } else {
        X = state32_ptr(L, 0, 0, sys); S = X; O = state32_ptr(L, 0, 1, sys);
        delta = 0.5 * L.dt; ta = 0.0; tb = 0.5 * L.dt;
    }
    __shared__ double Es[2];
    if (threadIdx.x < 2) Es[threadIdx.x] = field_E(c, threadIdx.x == 0 ? ta : tb);
    __syncthreads();
    if (m >= L.M1) return;
    const double kappa_d = (mode == 2) ? 0.5 * c.kappa_dt : c.kappa_dt;
    const double nu_d = 1.0 + 0.5 * delta, xi_d = 1.0 - 0.5 * delta;
    const double ph_d = L.phi[(size_t)sys * L.pitch + m];
    const float2 zero = make_float2(0.f, 0.f);
    const bool left = m > 0, right = m + 1 < L.M1;
    const size_t p = (size_t)L.pitch;
    const float2 lm = (n > 0 && left) ? S[(n - 1) * p + m - 1] : zero;     // (n-1, m-1)
    const float2 lp = (n > 0 && right) ? S[(n - 1) * p + m + 1] : zero;    // (n-1, m+1)
    const float2 um = (n < L.N && left) ? S[(n + 1) * p + m - 1] : zero;   // (n+1, m-1)
    const float2 up = (n < L.N && right) ? S[(n + 1) * p + m + 1] : zero;  // (n+1, m+1)
    const float2 w = X[n * p + m];
    float2 out;
    if (PREC == 1) {
        // fp64 arithmetic on the fp32 state: the same per-point expression as every fp64 kernel
        double2 lo, hi;
        lo.x = (double)lp.x - (double)lm.x; lo.y = (double)lp.y - (double)lm.y;
        if (n == 1) lo.x *= 2.0;                                           // chi(1) = 2, eq. (11)
        hi.x = (double)up.x - (double)um.x; hi.y = (double)up.y - (double)um.y;
        const double hba = __dmul_rn(__fma_rn(c.B, ph_d, Es[0]), 0.5 * delta);
        const double hbb = __dmul_rn(__fma_rn(c.B, ph_d, Es[1]), 0.5 * delta);
        const double src = __dmul_rn(cn_ptr(L, sys)[n], __dmul_rn(L.gm[(size_t)sys * L.pitch + m], delta));
        const double2 r = cn_point(make_double2((double)w.x, (double)w.y), lo, hi, (double)n, hba, hbb, src, kappa_d,
                                   xi_d, nu_d, nu_d * nu_d);
        out = make_float2((float)r.x, (float)r.y);                         // stored: rounded once
    } else {
        // fp32 throughout, eq. (28)-(37) in the order of the paper's loop nest (L294-303), one rounding per operation
        const float d = (float)delta, kap = (float)kappa_d, nu = (float)nu_d, xi = (float)xi_d;
        const float Ea = (float)Es[0], Eb = (float)Es[1], Bf = (float)c.B, ph = (float)ph_d, nf = (float)n;
        const float beta_a = __fadd_rn(Ea, __fmul_rn(Bf, ph));             // eq. (28)-(29)
        const float beta_b = __fadd_rn(Eb, __fmul_rn(Bf, ph));
        const float mu_a = __fmul_rn(__fmul_rn(__fmul_rn(nf, beta_a), d), 0.5f);   // x / 2 == x * 0.5 exactly
        const float mu_b = __fmul_rn(__fmul_rn(__fmul_rn(nf, beta_b), d), 0.5f);
        const float chi = (n == 1) ? 2.0f : 1.0f;                          // eq. (11)
        const float Bt = __fmul_rn(kap, __fadd_rn(__fsub_rn(__fsub_rn(up.y, um.y), lp.y), lm.y));            // eq. (31)
        const float At = __fmul_rn(kap, __fadd_rn(__fsub_rn(__fmul_rn(chi, __fsub_rn(lp.x, lm.x)), up.x), um.x));  // (30)
        const float src = __fmul_rn((float)cn_ptr(L, sys)[n], __fmul_rn((float)L.gm[(size_t)sys * L.pitch + m], d));
        const float g = __fadd_rn(__fadd_rn(__fsub_rn(__fmul_rn(w.x, xi), __fmul_rn(w.y, mu_a)), Bt), src);  // eq. (36)
        const float h = __fadd_rn(__fadd_rn(__fmul_rn(w.y, xi), __fmul_rn(w.x, mu_a)), At);                  // eq. (37)
        const float det = __fadd_rn(__fmul_rn(nu, nu), __fmul_rn(mu_b, mu_b));
        out.x = __fdiv_rn(__fsub_rn(__fmul_rn(g, nu), __fmul_rn(h, mu_b)), det);                             // eq. (32)
        out.y = __fdiv_rn(__fadd_rn(__fmul_rn(g, mu_b), __fmul_rn(h, nu)), det);                             // eq. (33), C2
    }
    if (n == 0) out.y = 0.f;                                               // b_0 == 0, eq. (23) / C3
    O[n * p + m] = out;
}

// host (fp64 arrays) <-> fp32 workspace state
__global__ void deinterleave32_kernel(const float2* __restrict__ z, double* __restrict__ a, double* __restrict__ b,
                                      int rows, int M1, int pitch) {
    const int n = blockIdx.y, m = blockIdx.x * blockDim.x + threadIdx.x;
    if (n >= rows || m >= M1) return;
    const float2 w = z[(size_t)n * pitch + m];
    a[(size_t)n * M1 + m] = (double)w.x;
    b[(size_t)n * M1 + m] = (double)w.y;
}

__global__ void interleave32_kernel(float2* __restrict__ z, const double* __restrict__ a, const double* __restrict__ b,
                                    int rows, int M1, int pitch) {
    const int n = blockIdx.y, m = blockIdx.x * blockDim.x + threadIdx.x;
    if (n >= rows || m >= pitch) return;
    float2 w = make_float2(0.f, 0.f);
    if (m < M1) {
        w.x = (float)a[(size_t)n * M1 + m];
        w.y = (n == 0) ? 0.f : (float)b[(size_t)n * M1 + m];
    }
    z[(size_t)n * pitch + m] = w;
}

}  // namespace bte
