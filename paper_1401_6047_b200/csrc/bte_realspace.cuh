// bte_realspace.cuh -- real-space-phi_x variant of the step (BASELINE config 0's "64 periodic
// phi_x points").  Not in the paper (its Fourier representation (7)-(8) turns the implicit solve into the 2x2 blocks
// of eq. 32-33); the same splitting of eq. (5) kept in real space (C22):
//   rhs_i = xi X_i - gamma_a (X_{i+1} - X_{i-1}) + kappa' sin(phi_x_i) (S_{i,m+1} - S_{i,m-1}) + f0_{i,m} delta
//   nu X'_i + gamma_b (X'_{i+1} - X'_{i-1}) = rhs_i,   i cyclic:  ONE CYCLIC TRIDIAGONAL SYSTEM PER phi_y ROW.
// Batched cyclic sweeps: one thread per phi_y lattice point m sweeps over i (Thomas algorithm on the tridiagonal
// part, the two corner entries by the Sherman-Morrison correction); f is stored [i][m] with m fastest, so every access
// of a sweep is coalesced across the threads of a warp.  In place: the forward sweep leaves the modified right-hand
// side where X was (old neighbours are carried in registers).
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

namespace bte {

struct RsObs {                 // device-resident observables and running sums
    double norm, v_dr, sum_v, sum_c, sum_s, window, edge_leak;
    unsigned int done, pad;
};

struct RsLayout {
    int K, M1, pitch;          // phi_x points, phi_y points, row pitch (multiple of 8)
    double dt, dx, dphi;
    double E_dc, E_omega, omega, B, kappa_scale;
    double norm_scale;         // sqrt(alpha) dx dphi  (eq. 6; eq. 18-19 for v_dr)
    double* f;                 // [grid 2][K][pitch]
    double* cprime;            // [K][pitch]   Thomas coefficients of the current half-update
    double* zvec;              // [K][pitch]   solution of T z = u (Sherman-Morrison)
    const double* ex;          // [K]  exp(mu cos phi_x_i) / (2 pi I0(mu)) sqrt(mu / (2 pi alpha))   (eq. 13, phi_x part)
    const double* sinx;        // [K]
    const double* gm;          // [pitch] exp(-mu phi_m^2 / 2)
    const double* phi;         // [pitch]
    double* partial;           // [blocks][2]
    RsObs* obs;
};

__device__ __forceinline__ double rs_warp_sum(double v) {
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
    return v;
}

__global__ void rs_init_kernel(RsLayout L) {
    const int m = blockIdx.x * blockDim.x + threadIdx.x, i = blockIdx.y;
    if (m >= L.pitch) return;
    L.f[(size_t)i * L.pitch + m] = (m < L.M1) ? L.ex[i] * L.gm[m] : 0.0;      // whole grid <- f0 (L99)
    if (blockIdx.x == 0 && i == 0 && threadIdx.x == 0) {
        RsObs z = {};
        *L.obs = z;
    }
}

// mode 0: whole grid (stencil: fractional), times k dt -> (k+1) dt;  mode 1: fractional grid (stencil: NEW whole grid),
// times (k+1/2) dt -> (k+3/2) dt;  mode 2: start-up, fractional <- T_{dt/2}(whole; stencil whole; 0 -> dt/2) (L202).
// do_sum: after a whole-grid update, fold norm / v_dr (and the running sums of eq. 17 if do_avg).
__global__ void __launch_bounds__(128) rs_half_update_kernel(RsLayout L, int mode, long long k, int do_avg) {
    __shared__ double red[2][4];
    __shared__ unsigned int s_last;
    const int m = blockIdx.x * blockDim.x + threadIdx.x;
    const int K = L.K;
    const size_t p = (size_t)L.pitch, G1 = (size_t)K * p;
    double* X = (mode == 0) ? L.f : L.f + G1;                    // grid written
    const double* S = (mode == 1) ? L.f : (mode == 0 ? L.f + G1 : L.f);   // stencil grid
    const double delta = (mode == 2) ? 0.5 * L.dt : L.dt;
    const double ta = (mode == 0) ? (double)k * L.dt : (mode == 1 ? ((double)k + 0.5) * L.dt : 0.0);
    const double tb = (mode == 0) ? ((double)k + 1.0) * L.dt : (mode == 1 ? ((double)k + 1.5) * L.dt : 0.5 * L.dt);
    double sa = 0.0, sv = 0.0;
    if (m < L.M1) {
        const double ph = L.phi[m];
        const double Ea = L.E_dc + L.E_omega * cos(L.omega * ta), Eb = L.E_dc + L.E_omega * cos(L.omega * tb);
        const double ga = (Ea + L.B * ph) * delta / (4.0 * L.dx), gb = (Eb + L.B * ph) * delta / (4.0 * L.dx);
        const double kap = L.kappa_scale * L.B * delta / (2.0 * L.dphi);
        const double nu = 1.0 + 0.5 * delta, xi = 1.0 - 0.5 * delta;
        const double gdt = L.gm[m] * delta;
        const bool left = m > 0, right = m + 1 < L.M1;
        const double* Xs = (mode == 2) ? L.f : X;                // start-up: the source is the whole grid
        // Sherman-Morrison for the two corner entries A[0][K-1] = -gb, A[K-1][0] = +gb:  A = T + u v^T with
        // u = (g0, 0, .., 0, gb), v = (1, 0, .., 0, -gb / g0), g0 = -nu;  T: diagonal nu except T_00 = nu - g0,
        // T_{K-1,K-1} = nu + gb (-gb) / g0, sub-diagonal -gb, super-diagonal +gb.
        const double g0 = -nu;
        const double x_first = Xs[m], x_last = Xs[(size_t)(K - 1) * p + m];
        double xm1 = x_last, xc = x_first, cp = 0.0, dp = 0.0, zp = 0.0;
        // forward sweep: right-hand sides rhs_i (eq. above) and u_i together
        for (int i = 0; i < K; ++i) {
            const double xp1 = (i + 1 < K) ? Xs[(size_t)(i + 1) * p + m] : x_first;
            const double sl = left ? S[(size_t)i * p + m - 1] : 0.0, sr = right ? S[(size_t)i * p + m + 1] : 0.0;
            const double rhs = xi * xc - ga * (xp1 - xm1) + kap * L.sinx[i] * (sr - sl) + L.ex[i] * gdt;
            const double u = (i == 0) ? g0 : (i == K - 1 ? gb : 0.0);
            const double diag = (i == 0) ? nu - g0 : (i == K - 1 ? nu + gb * gb / g0 : nu);   // nu - alpha beta / g0
            const double denom = diag + gb * cp;                 // sub-diagonal is -gb
            const double inv = 1.0 / denom;
            const double cn = gb * inv;
            dp = (rhs + gb * dp) * inv;
            zp = (u + gb * zp) * inv;
            X[(size_t)i * p + m] = dp;
            L.zvec[(size_t)i * p + m] = zp;
            L.cprime[(size_t)i * p + m] = cn;
            cp = cn;
            xm1 = xc; xc = xp1;
        }
        // back substitution for y (in X) and z
        double y = dp, z = zp;                                   // i = K-1
        const double y_last = y, z_last = z;
        for (int i = K - 2; i >= 0; --i) {
            const double c = L.cprime[(size_t)i * p + m];
            y = X[(size_t)i * p + m] - c * y;
            z = L.zvec[(size_t)i * p + m] - c * z;
            X[(size_t)i * p + m] = y;
            L.zvec[(size_t)i * p + m] = z;
        }
        const double vK = -gb / g0;                              // v = (1, 0, .., 0, vK)
        const double fact = (y + vK * y_last) / (1.0 + z + vK * z_last);
        for (int i = 0; i < K; ++i) {
            const double x = X[(size_t)i * p + m] - fact * L.zvec[(size_t)i * p + m];
            X[(size_t)i * p + m] = x;
            sa += x;
            sv += L.sinx[i] * x;
        }
    }
    if (mode != 0) return;
    // norm (eq. 6) and v_dr (eq. 18-19) of the new whole grid: block partials, last block folds in fixed order
    sa = rs_warp_sum(sa); sv = rs_warp_sum(sv);
    const int warp = threadIdx.x >> 5;
    if ((threadIdx.x & 31) == 0) { red[0][warp] = sa; red[1][warp] = sv; }
    __syncthreads();
    if (threadIdx.x == 0) {
        L.partial[2 * blockIdx.x] = (red[0][0] + red[0][1]) + (red[0][2] + red[0][3]);
        L.partial[2 * blockIdx.x + 1] = (red[1][0] + red[1][1]) + (red[1][2] + red[1][3]);
        __threadfence();
        s_last = (atomicAdd(&L.obs->done, 1u) + 1u == gridDim.x) ? 1u : 0u;
    }
    __syncthreads();
    if (s_last && threadIdx.x == 0) {
        __threadfence();
        double ta2 = 0.0, tv = 0.0;
        for (unsigned b = 0; b < gridDim.x; ++b) {
            ta2 += ((volatile double*)L.partial)[2 * b];
            tv += ((volatile double*)L.partial)[2 * b + 1];
        }
        RsObs* o = L.obs;
        o->norm = L.norm_scale * ta2;
        o->v_dr = L.norm_scale * tv;
        if (do_avg) {
            const double t = (double)(k + 1) * L.dt;
            double sn, cs;
            sincos(L.omega * t, &sn, &cs);
            o->sum_v += o->v_dr * L.dt; o->sum_c += o->v_dr * cs * L.dt; o->sum_s += o->v_dr * sn * L.dt;
            o->window += L.dt;
        }
        o->done = 0u;
    }
}

// ---- fast path: parallel cyclic reduction over phi_x (n_phix a power of two, <= RS_PCR_MAX_K) -----------------------------
// The matrix of one phi_y column is CIRCULANT (sub-diagonal a = -gamma_b, diagonal b = nu, super-diagonal c = +gamma_b,
// the same for every i), so parallel cyclic reduction needs the three numbers (a, b, c) per level and column only:
//   level h = 1, 2, 4, .., K/2:   alpha = -a / b, beta = -c / b,
//       d'_i = d_i + alpha d_{i-h} + beta d_{i+h}   (indices mod K),
//       a' = alpha a,   b' = b + alpha c + beta a,   c' = beta c;
//   after log2 K levels equation i couples x_i with x_{i +- K} = x_i:   x_i = d_i / (a + b + c).
// b' = nu + 2 gamma^2 / nu after the first level and |a'| + |c'| < b' from then on: no pivoting needed.
// A CTA of RS_PCR_MT warps takes a tile of RS_PCR_MT adjacent phi_y columns:
//   1. all threads form the right-hand sides of the tile in the coalesced (i, m) order of HBM (m fastest) and put them
//      into shared memory transposed (one column contiguous, column pitch K + 4: conflict-free both ways);
//   2. warp w takes column w into REGISTERS, lane l the K / 32 elements i = l mod 32, and reduces it there: the levels
//      h < 32 fetch d_{i -+ h} by warp shuffle (the source lane picks the register, r or r -+ 1, that the receiving lane's
//      wrap-around needs), the levels h >= 32 are register-to-register; no barrier inside the reduction;
//   3. all threads store the tile back in HBM order, folding norm and v_dr on the way.
// HBM traffic: X read once and written once, the stencil grid read once (+ the neighbour sector on either side of
// the tile): 24 B per point and half-update, no scratch arrays.
constexpr int RS_PCR_MT = 8;
constexpr int RS_PCR_T = 32 * RS_PCR_MT;
constexpr int RS_PCR_MAX_K = 1024;

__host__ __device__ constexpr size_t rs_pcr_smem(int K) { return (size_t)RS_PCR_MT * (K + 4) * sizeof(double); }

template <int K>
__global__ void __launch_bounds__(RS_PCR_T, K >= 1024 ? 2 : K >= 512 ? 3 : 4) rs_pcr_half_update_kernel(RsLayout L, int mode, long long k, int do_avg) {
    constexpr int R = K >= 32 ? K / 32 : 1;          // elements per lane
    constexpr int LN = K >= 32 ? 32 : K;             // lanes that hold elements
    constexpr int P = K + 4;                         // column pitch in shared memory: P mod 16 = 4 (K >= 16)
    constexpr int MT = RS_PCR_MT;
    constexpr int UNR = 4;                           // rows in flight per thread (5 loads each); 8 costs occupancy
    constexpr int ISTEP = RS_PCR_T / MT;             // = 32 rows per sweep of the CTA
    static_assert(ISTEP == 32 && (K & (K - 1)) == 0 && K >= 4, "tile shape");
    extern __shared__ double rs_sm[];
    __shared__ double red[2][MT];
    __shared__ unsigned int s_last;
    const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
    const size_t p = (size_t)L.pitch, G1 = (size_t)K * p;
    double* X = (mode == 0) ? L.f : L.f + G1;
    const double* S = (mode == 1) ? L.f : (mode == 0 ? L.f + G1 : L.f);
    const double* Xs = (mode == 2) ? L.f : X;
    const double delta = (mode == 2) ? 0.5 * L.dt : L.dt;
    const double ta = (mode == 0) ? (double)k * L.dt : (mode == 1 ? ((double)k + 0.5) * L.dt : 0.0);
    const double tb = (mode == 0) ? ((double)k + 1.0) * L.dt : (mode == 1 ? ((double)k + 1.5) * L.dt : 0.5 * L.dt);
    const double nu = 1.0 + 0.5 * delta, xi = 1.0 - 0.5 * delta;
    const int m0 = blockIdx.x * MT;
    const int ml = tid % MT, m = m0 + ml;            // this thread's column in the load / store phases (m < pitch)
    const int i0 = tid / MT;                         // and its first row
    // launched with programmatic stream serialization: the next half-update may become resident and form its constants
    // now; it waits (griddepcontrol.wait) for THIS grid to complete and flush before it touches f or the observables
    asm volatile("griddepcontrol.launch_dependents;");
    // 1. right-hand sides, transposed into shared memory
    {
        const double ph = L.phi[m];
        const double Ea = L.E_dc + L.E_omega * cos(L.omega * ta);
        const double ga = (Ea + L.B * ph) * delta / (4.0 * L.dx);
        const double kap = L.kappa_scale * L.B * delta / (2.0 * L.dphi);
        const double gdt = L.gm[m] * delta;
        asm volatile("griddepcontrol.wait;" ::: "memory");
        const bool left = m > 0 && m < L.M1, right = m + 1 < L.M1;
        const double* Xc = Xs + m;
        const double* Sc = S + m;
#pragma unroll UNR
        for (int j = 0; j < R; ++j) {
            const int i = i0 + ISTEP * j;
            if (K >= 32 || i < K) {
                const double sl = left ? Sc[(size_t)i * p - 1] : 0.0, sr = right ? Sc[(size_t)i * p + 1] : 0.0;
                const double xp1 = Xc[(size_t)((i + 1) & (K - 1)) * p], xm1 = Xc[(size_t)((i - 1) & (K - 1)) * p];
                rs_sm[ml * P + i] = xi * Xc[(size_t)i * p] - ga * (xp1 - xm1) + kap * L.sinx[i] * (sr - sl) + L.ex[i] * gdt;
            }
        }
    }
    __syncthreads();
    // 2. warp w: parallel cyclic reduction of column m0 + w in registers
    {
        double* col = rs_sm + warp * P;
        double d[R];
#pragma unroll
        for (int r = 0; r < R; ++r) d[r] = (K >= 32 || lane < K) ? col[lane + 32 * r] : 0.0;
        const double ph = L.phi[m0 + warp];
        const double Eb = L.E_dc + L.E_omega * cos(L.omega * tb);
        const double gb = (Eb + L.B * ph) * delta / (4.0 * L.dx);
        double a = -gb, b = nu, c = gb;
#pragma unroll
        for (int h = 1; h < LN; h <<= 1) {                      // neighbours in other lanes
            const double rb = 1.0 / b, alpha = -a * rb, beta = -c * rb;
            const bool wrap_up = lane >= LN - h, wrap_dn = lane < h;   // as a SOURCE: the receiver wrapped around the column
            const int src_up = (lane - h) & (LN - 1), src_dn = (lane + h) & (LN - 1);
            double dn[R];
#pragma unroll
            for (int r = 0; r < R; ++r) {
                const double send_up = wrap_up ? d[(r + R - 1) % R] : d[r];      // element i - h of the receiver
                const double send_dn = wrap_dn ? d[(r + 1) % R] : d[r];          // element i + h of the receiver
                const double up = __shfl_sync(0xffffffffu, send_up, src_up);
                const double dw = __shfl_sync(0xffffffffu, send_dn, src_dn);
                dn[r] = d[r] + alpha * up + beta * dw;
            }
#pragma unroll
            for (int r = 0; r < R; ++r) d[r] = dn[r];
            const double a2 = alpha * a, b2 = b + alpha * c + beta * a, c2 = beta * c;
            a = a2; b = b2; c = c2;
        }
#pragma unroll
        for (int q = 1; q < R; q <<= 1) {                       // h = 32 q: neighbours in this lane's own registers
            const double rb = 1.0 / b, alpha = -a * rb, beta = -c * rb;
            double dn[R];
#pragma unroll
            for (int r = 0; r < R; ++r) dn[r] = d[r] + alpha * d[(r + R - q) % R] + beta * d[(r + q) % R];
#pragma unroll
            for (int r = 0; r < R; ++r) d[r] = dn[r];
            const double a2 = alpha * a, b2 = b + alpha * c + beta * a, c2 = beta * c;
            a = a2; b = b2; c = c2;
        }
        const double scale = 1.0 / (a + b + c);                 // x_i = d_i / (a + b + c)
#pragma unroll
        for (int r = 0; r < R; ++r)
            if (K >= 32 || lane < K) col[lane + 32 * r] = d[r] * scale;
    }
    __syncthreads();
    // 3. store in HBM order; norm (eq. 6) and v_dr (eq. 18-19) of a new whole grid
    double sa = 0.0, sv = 0.0;
    if (m < L.M1) {
#pragma unroll 4
        for (int j = 0; j < R; ++j) {
            const int i = i0 + ISTEP * j;
            if (K >= 32 || i < K) {
                const double x = rs_sm[ml * P + i];
                X[(size_t)i * p + m] = x;
                sa += x;
                sv += L.sinx[i] * x;
            }
        }
    }
    if (mode != 0) return;
    sa = rs_warp_sum(sa); sv = rs_warp_sum(sv);
    if (lane == 0) { red[0][warp] = sa; red[1][warp] = sv; }
    __syncthreads();
    if (tid == 0) {
        double qa = 0.0, qv = 0.0;
        for (int w = 0; w < MT; ++w) { qa += red[0][w]; qv += red[1][w]; }
        L.partial[2 * blockIdx.x] = qa;
        L.partial[2 * blockIdx.x + 1] = qv;
        __threadfence();
        s_last = (atomicAdd(&L.obs->done, 1u) + 1u == gridDim.x) ? 1u : 0u;
    }
    __syncthreads();
    if (s_last && warp == 0) {                                 // fixed-order fold: lane-strided sums, then the shuffle tree
        __threadfence();
        double qa = 0.0, qv = 0.0;
        for (unsigned bq = lane; bq < gridDim.x; bq += 32) {
            qa += __ldcg(L.partial + 2 * bq);
            qv += __ldcg(L.partial + 2 * bq + 1);
        }
        qa = rs_warp_sum(qa); qv = rs_warp_sum(qv);
        if (lane == 0) {
            RsObs* o = L.obs;
            o->norm = L.norm_scale * qa;
            o->v_dr = L.norm_scale * qv;
            if (do_avg) {
                const double t = (double)(k + 1) * L.dt;
                double sn, cs;
                sincos(L.omega * t, &sn, &cs);
                o->sum_v += o->v_dr * L.dt; o->sum_c += o->v_dr * cs * L.dt; o->sum_s += o->v_dr * sn * L.dt;
                o->window += L.dt;
            }
            o->done = 0u;
        }
    }
}

using RsKernel = void (*)(RsLayout, int, long long, int);
inline RsKernel rs_pcr_kernel_for(int K) {
    switch (K) {
        case 4: return rs_pcr_half_update_kernel<4>;
        case 8: return rs_pcr_half_update_kernel<8>;
        case 16: return rs_pcr_half_update_kernel<16>;
        case 32: return rs_pcr_half_update_kernel<32>;
        case 64: return rs_pcr_half_update_kernel<64>;
        case 128: return rs_pcr_half_update_kernel<128>;
        case 256: return rs_pcr_half_update_kernel<256>;
        case 512: return rs_pcr_half_update_kernel<512>;
        case 1024: return rs_pcr_half_update_kernel<1024>;
        default: return nullptr;
    }
}

}  // namespace bte
