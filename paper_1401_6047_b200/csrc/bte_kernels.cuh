// bte_kernels.cuh -- the simple sm_100a kernels of libbte_b200 (the production step kernels live in
// bte_sweep.cuh and bte_resident.cuh and include this file).
//
//   init_state_kernel        a_h = a^(0) = c_n g_m, b_h = 0                       (eq. 15)
//   half_update_kernel       one application of T (eq. 38) to one grid, one thread per lattice point: the
//                            "split" variant of the step (two launches per step, 96 B/point; cross-check of the
//                            production kernels) and the start-up z^{1/2} (L202)
//   reduce_finalize_kernel   norm / v_dr / running sums for the split variants and after init / set_state
//                            (multi-block, deterministic last-block fold; templated on the state type)
//   fused_step_kernel        whole + fractional update in ONE sweep over a 2-D tile grid (variant 2, cross-check):
//                            each CTA marches a strip of phi_y columns over a chunk of harmonics, rows staged
//                            through a shared-memory ring by cp.async (zero-fill = boundary conditions 22-23)
//   (de)interleave kernels   host <-> workspace state exchange
//   pdf_kernel               f(phi_x, phi_y) of eq. (8) from the coefficients
#pragma once
#include "bte_device.cuh"

namespace bte {

// ------------------------------------------------------------------------------------------------
// small helpers
// ------------------------------------------------------------------------------------------------
__device__ __forceinline__ void cp_async16_zfill(void* smem_dst, const void* gmem_src, bool valid) {
    const unsigned s = (unsigned)__cvta_generic_to_shared(smem_dst);
    const int n = valid ? 16 : 0;   // src-size 0 => 16 bytes of zeros are written (ghost cells, eq. 22-23)
    asm volatile("cp.async.cg.shared.global [%0], [%1], 16, %2;\n" ::"r"(s), "l"(gmem_src), "r"(n)
                 : "memory");
}
__device__ __forceinline__ void cp_async_commit() { asm volatile("cp.async.commit_group;\n" ::: "memory"); }
template <int N>
__device__ __forceinline__ void cp_async_wait() {
    asm volatile("cp.async.wait_group %0;\n" ::"n"(N) : "memory");
}

__device__ __forceinline__ double warp_sum(double v) {
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
    return v;
}

// Fold of the per-strip partial sums and the per-step bookkeeping of one system, executed by warp 0 of
// the last block of that system to finish (fixed summation order => deterministic).
// eq. (12), (20) by the rectangle rule (C10); running sums of eq. (17) for steps k+1 > avg_start (C9).
//   mode 0: observables only (after init / set_state)
//   mode 1: observables + running sums + step counter k <- k+1, live buffer toggled
//   mode 2: observables + running sums; the step counter is advanced by the caller
__device__ __forceinline__ void fold_and_advance(const Layout& L, int sys, int n_partials, long long k,
                                                 int mode) {
    const int lane = threadIdx.x & 31;
    const volatile double* part = L.partial + (size_t)sys * L.pitch * 2;
    double sa = 0.0, sb = 0.0;
    for (int s = lane; s < n_partials; s += 32) {
        sa += part[2 * s];
        sb += part[2 * s + 1];
    }
    sa = warp_sum(sa);
    sb = warp_sum(sb);
    if (lane == 0) {
        const SysConst c = L.sc[sys];
        SysState* st = L.ss + sys;
        const double norm = c.norm_scale * sa;
        const double v = c.v_scale * sb;
        st->norm = norm;
        st->v_dr = v;
        st->edge_leak = ((volatile double*)st->edge)[0] + ((volatile double*)st->edge)[1];
        if (mode != 0) {
            const long long k1 = k + 1;
            if (k1 > c.avg_start_step) {
                const double t = (double)k1 * L.dt;
                double sn, cs;
                sincos(c.omega * t, &sn, &cs);
                st->sum_v += v * L.dt;
                st->sum_c += v * cs * L.dt;
                st->sum_s += v * sn * L.dt;
                st->window += L.dt;
            }
            if (mode == 1) { st->k = k1; st->buf ^= 1; }
        }
        st->done = 0u;
        __threadfence();
    }
}

// ------------------------------------------------------------------------------------------------
// init: whole grid of buffer 0 <- equilibrium (eq. 15); resets the bookkeeping
// ------------------------------------------------------------------------------------------------
__global__ void init_state_kernel(Layout L) {
    const int sys = blockIdx.z, n = blockIdx.y;
    const int m = blockIdx.x * blockDim.x + threadIdx.x;
    if (blockIdx.x == 0 && n == 0 && threadIdx.x == 0) {
        SysState z = {};
        L.ss[sys] = z;
    }
    if (m >= L.pitch) return;
    double2 w = make_double2(0.0, 0.0);
    if (m < L.M1) w.x = cn_ptr(L, sys)[n] * L.gm[(size_t)sys * L.pitch + m];
    double2* H = state_ptr(L, 0, 0, sys);
    H[(size_t)n * L.pitch + m] = w;
}

// ------------------------------------------------------------------------------------------------
// split variant / start-up: one application of T to one grid, one thread per lattice point
//   mode 0: whole grid      H[nxt] <- T_dt (H[cur]; stencil F[cur];  t_k,       t_{k+1})     eq. (40)
//   mode 1: fractional grid F[nxt] <- T_dt (F[cur]; stencil H[nxt];  t_{k+1/2}, t_{k+3/2})   eq. (41)
//   mode 2: start-up        F[0]   <- T_{dt/2}(H[0]; stencil H[0];   0,         dt/2)        L202, C6
// ------------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(128) half_update_kernel(Layout L, int mode) {
    const int sys = blockIdx.z, n = blockIdx.y;
    const int m = blockIdx.x * blockDim.x + threadIdx.x;
    const SysConst c = L.sc[sys];
    const long long k = (mode == 2) ? 0 : L.ss[sys].k;
    if (mode != 2 && c.n_steps_total > 0 && k >= c.n_steps_total) return;   // frozen system
    const int cur = (mode == 2) ? 0 : L.ss[sys].buf, nxt = cur ^ 1;
    const double2 *X, *S;
    double2* O;
    double delta, ta, tb;
    if (mode == 0) {
        X = state_ptr(L, cur, 0, sys); S = state_ptr(L, cur, 1, sys); O = state_ptr(L, nxt, 0, sys);
        delta = L.dt; ta = (double)k * L.dt; tb = ((double)k + 1.0) * L.dt;
    } else if (mode == 1) {
        X = state_ptr(L, cur, 1, sys); S = state_ptr(L, nxt, 0, sys); O = state_ptr(L, nxt, 1, sys);
        delta = L.dt; ta = ((double)k + 0.5) * L.dt; tb = ((double)k + 1.5) * L.dt;
    } else {
        X = state_ptr(L, 0, 0, sys); S = X; O = state_ptr(L, 0, 1, sys);
        delta = 0.5 * L.dt; ta = 0.0; tb = 0.5 * L.dt;
    }
    __shared__ double Es[2];
    if (threadIdx.x < 2) Es[threadIdx.x] = field_E(c, threadIdx.x == 0 ? ta : tb);
    __syncthreads();
    if (m >= L.M1) return;
    const double kappa = (mode == 2) ? 0.5 * c.kappa_dt : c.kappa_dt;
    const double nu = 1.0 + 0.5 * delta, xi = 1.0 - 0.5 * delta;
    const double ph = L.phi[(size_t)sys * L.pitch + m];
    const double hba = __dmul_rn(__fma_rn(c.B, ph, Es[0]), 0.5 * delta);
    const double hbb = __dmul_rn(__fma_rn(c.B, ph, Es[1]), 0.5 * delta);
    const double src = __dmul_rn(cn_ptr(L, sys)[n], __dmul_rn(L.gm[(size_t)sys * L.pitch + m], delta));
    const double2 zero = make_double2(0.0, 0.0);
    const bool left = m > 0, right = m + 1 < L.M1;
    const size_t p = (size_t)L.pitch;
    double2 lo = zero, hi = zero;
    if (n > 0) {
        const double2 l = left ? S[(n - 1) * p + m - 1] : zero;
        const double2 r = right ? S[(n - 1) * p + m + 1] : zero;
        lo.x = r.x - l.x; lo.y = r.y - l.y;
        if (n == 1) lo.x *= 2.0;   // chi(1) = 2, eq. (11)
    }
    if (n < L.N) {
        const double2 l = left ? S[(n + 1) * p + m - 1] : zero;
        const double2 r = right ? S[(n + 1) * p + m + 1] : zero;
        hi.x = r.x - l.x; hi.y = r.y - l.y;
    }
    double2 w = cn_point(X[n * p + m], lo, hi, (double)n, hba, hbb, src, kappa, xi, nu, nu * nu);
    if (n == 0) w.y = 0.0;   // b_0 == 0, eq. (23) / C3
    O[n * p + m] = w;
}

// Sums row 0 (a) and row 1 (b) of the whole grid in buffer (buf ^ advance) and folds.  Used by the split variants
// (advance = 1) and after init / set_state (advance = 0).  grid = (RED_BLOCKS-or-fewer column chunks, n_batch);
// the last block of a system to finish folds the per-warp partial sums in fixed order (deterministic).
// E2 = double2 (fp64 state) or float2 (fp32 state, bte_lowprec.cuh); sums accumulate in fp64 either way.
constexpr int RED_BLOCKS = 64;

template <class E2>
__device__ __forceinline__ E2* state_ptr_t(const Layout& L, int buf, int grid, int sys) {
    return (E2*)L.state + (((size_t)buf * 2 + grid) * L.n_batch + sys) * grid_points(L) + (size_t)GHOST * L.pitch;
}

template <class E2>
__global__ void __launch_bounds__(256) reduce_finalize_kernel(Layout L, int advance) {
    __shared__ unsigned int s_last;
    const int sys = blockIdx.y;
    const SysConst c = L.sc[sys];
    const long long k = L.ss[sys].k;
    if (advance && c.n_steps_total > 0 && k >= c.n_steps_total) return;
    const int buf = L.ss[sys].buf ^ (advance ? 1 : 0);
    const E2* H = state_ptr_t<E2>(L, buf, 0, sys);
    const int chunk = (L.M1 + gridDim.x - 1) / gridDim.x;
    const int m0 = blockIdx.x * chunk, m1 = min(L.M1, m0 + chunk);
    double sa = 0.0, sb = 0.0;
    for (int m = m0 + threadIdx.x; m < m1; m += blockDim.x) {
        sa += (double)H[m].x;
        sb += (double)H[(size_t)L.pitch + m].y;   // N >= 1 is enforced by bte_create
    }
    sa = warp_sum(sa);
    sb = warp_sum(sb);
    double* part = L.partial + (size_t)sys * L.pitch * 2;
    const int warp = threadIdx.x >> 5, slot = blockIdx.x * 8 + warp;     // 8 warps per block
    if ((threadIdx.x & 31) == 0) {
        part[2 * slot] = sa;
        part[2 * slot + 1] = sb;
    }
    if (blockIdx.x == 0 && threadIdx.x == 0) L.ss[sys].edge[0] = fabs((double)H[(size_t)L.pitch].y);
    if (blockIdx.x == gridDim.x - 1 && threadIdx.x == 0) L.ss[sys].edge[1] = fabs((double)H[(size_t)L.pitch + L.M1 - 1].y);
    __threadfence();
    __syncthreads();
    if (threadIdx.x == 0) s_last = (atomicAdd(&L.ss[sys].done, 1u) + 1u == gridDim.x) ? 1u : 0u;
    __syncthreads();
    if (s_last && warp == 0) {
        __threadfence();
        fold_and_advance(L, sys, (int)gridDim.x * 8, k, advance ? 1 : 0);
    }
}

// ------------------------------------------------------------------------------------------------
// fused step: whole + fractional update in one sweep (eq. 40-41), ping-pong buffers
//
// CTA (strip s, chunk q, system z): output columns [c0, c0+W), W = T-2, rows [r0, r0+Lr).
// Thread i owns column c = c0-1+i (threads 0 and T-1 are halo columns: they compute the new whole grid
// there, redundantly with the neighbouring strip, but store nothing).
// Iteration u = 0 .. Lr+4 (one __syncthreads each):
//   - row r0-2+u of F_old (T+2 columns) and of H_old (T columns) has arrived in ring slot u % R
//   - dF(row r0-2+u) = F_old[.,m+1] - F_old[.,m-1]                                (registers)
//   - H_new[jH = r0-3+u] from H_old[jH], dF(jH-1), dF(jH+1)  -> global + 2-slot smem ring
//   - dH(jH-1) from the ring row written one iteration ago
//   - F_new[jF = jH-2] from F_old[jF], dH(jF-1), dH(jF+1)    -> global
// Rows outside [0, N] and columns outside [0, M] are zero (cp.async zero-fill / predicates): eq. (22)-(23).
// ------------------------------------------------------------------------------------------------
template <int T, int D>
struct FusedCfg {
    static constexpr int W = T - 2;       // output columns per strip
    static constexpr int R = D + 5;       // ring slots: rows u-3..u live, u+1..u+D+1 in flight
    static constexpr int FCOLS = T + 2;   // F_old columns c0-2 .. c0+W+1
    static constexpr size_t smem_bytes = sizeof(double2) * ((size_t)R * (FCOLS + T) + 2 * T);
};

template <int T, int D>
__global__ void __launch_bounds__(T) fused_step_kernel(Layout L, int rows_per_chunk) {
    using Cfg = FusedCfg<T, D>;
    constexpr int W = Cfg::W, R = Cfg::R, FCOLS = Cfg::FCOLS;
    extern __shared__ double2 smem[];
    double2* Fring = smem;                          // [R][FCOLS]
    double2* Hring = smem + (size_t)R * FCOLS;      // [R][T]
    double2* Hn = Hring + (size_t)R * T;            // [2][T]
    __shared__ double Es[4];
    __shared__ double red[2][T / 32];
    __shared__ unsigned int s_last;

    const int sys = blockIdx.z, strip = blockIdx.x, chunk = blockIdx.y;
    const SysConst c = L.sc[sys];
    const long long k = L.ss[sys].k;
    if (c.n_steps_total > 0 && k >= c.n_steps_total) return;   // frozen system: nothing to do
    const int cur = L.ss[sys].buf, nxt = cur ^ 1;
    const double2* __restrict__ Hold = state_ptr(L, cur, 0, sys);
    const double2* __restrict__ Fold = state_ptr(L, cur, 1, sys);
    double2* __restrict__ Hnew = state_ptr(L, nxt, 0, sys);
    double2* __restrict__ Fnew = state_ptr(L, nxt, 1, sys);

    const int i = threadIdx.x;
    const int c0 = strip * W, r0 = chunk * rows_per_chunk;
    const int Lr = min(rows_per_chunk, L.N + 1 - r0);
    const int col = c0 - 1 + i;
    const bool col_valid = (col >= 0) && (col < L.M1);
    const bool owner = (i >= 1) && (i <= W) && col_valid;
    const size_t pitch = (size_t)L.pitch;

    // field at the four half-step times of this step: t_k, t_{k+1/2}, t_{k+1}, t_{k+3/2}  (C14)
    if (i < 4) Es[i] = field_E(c, ((double)k + 0.5 * (double)i) * L.dt);

    // load unit u = row r0-2+u of F_old and H_old -> ring slot
    auto issue = [&](int u, int slot) {
        const int row = r0 - 2 + u;
        const bool row_ok = (row >= 0) && (row <= L.N) && (u <= Lr + 3);
        const size_t roff = (size_t)(row_ok ? row : 0) * pitch;
        {
            const int cf = c0 - 2 + i;
            const bool ok = row_ok && cf >= 0 && cf < L.M1;
            cp_async16_zfill(Fring + (size_t)slot * FCOLS + i, Fold + (ok ? roff + cf : 0), ok);
        }
        if (i < 2) {
            const int cf = c0 - 2 + T + i;
            const bool ok = row_ok && cf < L.M1;
            cp_async16_zfill(Fring + (size_t)slot * FCOLS + T + i, Fold + (ok ? roff + cf : 0), ok);
        }
        if (u >= 1 && u <= Lr + 2) {   // H_old rows r0-1 .. r0+Lr
            const bool ok = row_ok && col_valid;
            cp_async16_zfill(Hring + (size_t)slot * T + i, Hold + (ok ? roff + col : 0), ok);
        }
        cp_async_commit();
    };

#pragma unroll
    for (int u = 0; u <= D; ++u) issue(u, u);   // prologue: units 0..D in flight

    const double ph = col_valid ? L.phi[(size_t)sys * L.pitch + col] : 0.0;
    const double gdt = col_valid ? __dmul_rn(L.gm[(size_t)sys * L.pitch + col], L.dt) : 0.0;
    const double* __restrict__ cn = cn_ptr(L, sys);
    const double kappa = c.kappa_dt;
    const double nu = 1.0 + 0.5 * L.dt, xi = 1.0 - 0.5 * L.dt, nu2 = nu * nu;
    __syncthreads();   // Es visible
    const double hd = 0.5 * L.dt;
    const double hbHa = __dmul_rn(__fma_rn(c.B, ph, Es[0]), hd);   // whole grid: explicit time t_k
    const double hbHb = __dmul_rn(__fma_rn(c.B, ph, Es[2]), hd);   //             implicit time t_{k+1}
    const double hbFa = __dmul_rn(__fma_rn(c.B, ph, Es[1]), hd);   // fractional grid: t_{k+1/2}
    const double hbFb = __dmul_rn(__fma_rn(c.B, ph, Es[3]), hd);   //                  t_{k+3/2}

    const double2 zero = make_double2(0.0, 0.0);
    double2 dF1 = zero, dF2 = zero;   // dF of the rows that arrived 1 and 2 iterations ago
    double2 dH1 = zero, dH2 = zero;   // dH of the rows formed 1 and 2 iterations ago
    double acc_a0 = 0.0, acc_b1 = 0.0;
    int slot_u = 0;          // u % R
    int slot_issue = D + 1;  // (u + D + 1) % R
    const int n_iter = Lr + 5;
    for (int u = 0; u < n_iter; ++u) {
        cp_async_wait<D>();   // this thread's copies of unit u have landed
        __syncthreads();      // ... everybody's; also orders the Hn ring and frees slot (u-4) % R
        issue(u + D + 1, slot_issue);

        // dF of the arriving row (row 0 pre-doubled in its a-component: chi(1) = 2, eq. 11)
        const double2* frow = Fring + (size_t)slot_u * FCOLS;
        double2 dF0;
        {
            const double2 l = frow[i], r = frow[i + 2];
            dF0.x = __dsub_rn(r.x, l.x); dF0.y = __dsub_rn(r.y, l.y);
            if (r0 - 2 + u == 0) dF0.x *= 2.0;
        }
        // whole grid, row jH (eq. 40)
        const int jH = r0 - 3 + u;
        double2 hn = zero;
        if (u >= 2 && u <= Lr + 3 && jH >= 0 && jH <= L.N && col_valid) {
            const int slot_h = (slot_u == 0) ? R - 1 : slot_u - 1;   // unit u-1 holds row jH
            const double2 w = Hring[(size_t)slot_h * T + i];
            hn = cn_point(w, dF2, dF0, (double)jH, hbHa, hbHb, __dmul_rn(cn[jH], gdt), kappa, xi, nu, nu2);
            if (jH == 0) hn.y = 0.0;   // b_0 == 0
            if (owner && jH >= r0 && jH < r0 + Lr) {
                Hnew[(size_t)jH * pitch + col] = hn;
                if (jH == 0) acc_a0 = hn.x;
                if (jH == 1) {
                    acc_b1 = hn.y;
                    if (col == 0) L.ss[sys].edge[0] = fabs(hn.y);
                    if (col == L.M1 - 1) L.ss[sys].edge[1] = fabs(hn.y);
                }
            }
        }
        Hn[(u & 1) * T + i] = hn;
        // dH of row jH-1, written one iteration ago (visible since this iteration's barrier)
        double2 dH0 = zero;
        if (i >= 1 && i <= W) {
            const double2* hrow = Hn + ((u + 1) & 1) * T;
            const double2 l = hrow[i - 1], r = hrow[i + 1];
            dH0.x = __dsub_rn(r.x, l.x); dH0.y = __dsub_rn(r.y, l.y);
            if (jH - 1 == 0) dH0.x *= 2.0;
        }
        // fractional grid, row jF = jH-2 (eq. 41): stencil from the NEW whole grid (C5)
        const int jF = jH - 2;
        if (owner && jF >= r0 && jF < r0 + Lr) {
            int slot_f = slot_u - 3; if (slot_f < 0) slot_f += R;    // unit u-3 holds row jF
            const double2 w = Fring[(size_t)slot_f * FCOLS + i + 1];
            double2 fn = cn_point(w, dH2, dH0, (double)jF, hbFa, hbFb, __dmul_rn(cn[jF], gdt), kappa, xi, nu, nu2);
            if (jF == 0) fn.y = 0.0;
            Fnew[(size_t)jF * pitch + col] = fn;
        }
        dF2 = dF1; dF1 = dF0;
        dH2 = dH1; dH1 = dH0;
        slot_u = (slot_u + 1 == R) ? 0 : slot_u + 1;
        slot_issue = (slot_issue + 1 == R) ? 0 : slot_issue + 1;
    }
    cp_async_wait<0>();

    // per-strip partial sums of row 0 (a) and row 1 (b) -> eq. (12), (20)
    if (chunk == 0) {
        const double sa = warp_sum(acc_a0), sb = warp_sum(acc_b1);
        if ((i & 31) == 0) { red[0][i >> 5] = sa; red[1][i >> 5] = sb; }
        __syncthreads();
        if (i == 0) {
            double ta = 0.0, tb = 0.0;
#pragma unroll
            for (int w = 0; w < T / 32; ++w) { ta += red[0][w]; tb += red[1][w]; }
            double* part = L.partial + ((size_t)sys * L.pitch + strip) * 2;
            part[0] = ta;
            part[1] = tb;
        }
    }
    // last block of this system to finish folds the partials and advances the step counter
    __threadfence();
    __syncthreads();
    if (i == 0) {
        const unsigned int total = gridDim.x * gridDim.y;
        const unsigned int prev = atomicAdd(&L.ss[sys].done, 1u);
        s_last = (prev + 1u == total) ? 1u : 0u;
    }
    __syncthreads();
    if (s_last && i < 32) {
        __threadfence();
        fold_and_advance(L, sys, (int)gridDim.x, k, 1);
    }
}

// ------------------------------------------------------------------------------------------------
// host <-> workspace state exchange: interleaved (a,b)[N+1][pitch]  <->  a[(N+1) M1], b[(N+1) M1]
// ------------------------------------------------------------------------------------------------
__global__ void deinterleave_kernel(const double2* __restrict__ z, double* __restrict__ a,
                                    double* __restrict__ b, int rows, int M1, int pitch) {
    const int n = blockIdx.y, m = blockIdx.x * blockDim.x + threadIdx.x;
    if (n >= rows || m >= M1) return;
    const double2 w = z[(size_t)n * pitch + m];
    a[(size_t)n * M1 + m] = w.x;
    b[(size_t)n * M1 + m] = w.y;
}

__global__ void interleave_kernel(double2* __restrict__ z, const double* __restrict__ a,
                                  const double* __restrict__ b, int rows, int M1, int pitch) {
    const int n = blockIdx.y, m = blockIdx.x * blockDim.x + threadIdx.x;
    if (n >= rows || m >= pitch) return;
    double2 w = make_double2(0.0, 0.0);
    if (m < M1) {
        w.x = a[(size_t)n * M1 + m];
        w.y = (n == 0) ? 0.0 : b[(size_t)n * M1 + m];   // b_0 == 0, eq. (23)
    }
    z[(size_t)n * pitch + m] = w;
}

// ---- whole-batch forms (bte_get_state_batch / bte_set_state_batch): no host round trip for the buffer flags ------
// Systems whose live buffer is 1 are copied into buffer 0 (both grids, ghost rows and pad columns included) ...
template <class E2>
__global__ void copy_live_to_buffer0_kernel(Layout L) {
    const int sys = blockIdx.z, grid = blockIdx.y;
    if (L.ss[sys].buf == 0) return;
    const size_t per = grid_points(L);
    const E2* src = (const E2*)L.state + ((size_t)(2 + grid) * L.n_batch + sys) * per;
    E2* dst = (E2*)L.state + ((size_t)grid * L.n_batch + sys) * per;
    for (size_t e = (size_t)blockIdx.x * blockDim.x + threadIdx.x; e < per; e += (size_t)gridDim.x * blockDim.x) dst[e] = src[e];
}
// ... and then every flag says 0.
__global__ void clear_buffer_flags_kernel(Layout L) {
    const int s = blockIdx.x * blockDim.x + threadIdx.x;
    if (s < L.n_batch) L.ss[s].buf = 0;
}
// buffer 0 -> de-interleaved a | b in rows 0..N of the same system and grid of buffer 1 (dead between steps)
__global__ void deinterleave_batch_kernel(Layout L, int grid) {
    const int sys = blockIdx.z, n = blockIdx.y, m = blockIdx.x * blockDim.x + threadIdx.x;
    if (m >= L.M1) return;
    const size_t cnt = (size_t)(L.N + 1) * L.M1;
    const double2 w = state_ptr(L, 0, grid, sys)[(size_t)n * L.pitch + m];
    double* stage = (double*)state_ptr(L, 1, grid, sys);
    stage[(size_t)n * L.M1 + m] = w.x;
    stage[cnt + (size_t)n * L.M1 + m] = w.y;
}
// a | b staged in buffer 1 -> interleaved state in buffer 0 (pad columns zero, b_0 = 0)
__global__ void interleave_batch_kernel(Layout L, int grid) {
    const int sys = blockIdx.z, n = blockIdx.y, m = blockIdx.x * blockDim.x + threadIdx.x;
    if (m >= L.pitch) return;
    const size_t cnt = (size_t)(L.N + 1) * L.M1;
    const double* stage = (const double*)state_ptr(L, 1, grid, sys);
    double2 w = make_double2(0.0, 0.0);
    if (m < L.M1) {
        w.x = stage[(size_t)n * L.M1 + m];
        w.y = (n == 0) ? 0.0 : stage[cnt + (size_t)n * L.M1 + m];   // b_0 == 0, eq. (23)
    }
    state_ptr(L, 0, grid, sys)[(size_t)n * L.pitch + m] = w;
}

// ------------------------------------------------------------------------------------------------
// the distribution function itself: f(phi_x, phi_y) = sum_n a_n cos(n phi_x) + b_n sin(n phi_x)
// (eq. 8) on K equidistant phi_x_i = -pi + 2 pi i / K, for every phi_y lattice point; f is [K][M1], m fastest.
// n phi_x_i = -n pi + 2 pi (n i mod K) / K exactly, so cos(n phi_x_i) = (-1)^n cos(2 pi j / K) with j = n i mod K
// kept in integers: one K-entry table per CTA, no argument reduction error however large n is.
// Thread = one phi_y column x KT values of phi_x; rows are read coalesced, each (a, b) once per KT outputs.
// ------------------------------------------------------------------------------------------------
template <int KT>
__global__ void __launch_bounds__(128) pdf_kernel(const double2* __restrict__ z, double* __restrict__ f, int rows,
                                                  int M1, int pitch, int K) {
    extern __shared__ double tab[];          // cos(2 pi j / K), sin(2 pi j / K), j = 0..K-1
    double* cs = tab;
    double* sn = tab + K;
    for (int j = threadIdx.x; j < K; j += blockDim.x) sincospi(2.0 * (double)j / (double)K, sn + j, cs + j);
    __syncthreads();
    const int m = blockIdx.x * blockDim.x + threadIdx.x;
    const int i0 = blockIdx.y * KT;
    if (m >= M1) return;
    double acc[KT];
    int jn[KT];                              // n * i mod K
#pragma unroll
    for (int t = 0; t < KT; ++t) { acc[t] = 0.0; jn[t] = 0; }
    for (int n = 0; n < rows; ++n) {
        double2 w = z[(size_t)n * pitch + m];
        if (n & 1) { w.x = -w.x; w.y = -w.y; }            // (-1)^n
#pragma unroll
        for (int t = 0; t < KT; ++t) {
            acc[t] = __fma_rn(w.x, cs[jn[t]], __fma_rn(w.y, sn[jn[t]], acc[t]));
            jn[t] += (i0 + t < K) ? i0 + t : 0;             // chunk tail beyond K: index stays 0, value unused
            if (jn[t] >= K) jn[t] -= K;
        }
    }
#pragma unroll
    for (int t = 0; t < KT; ++t)
        if (i0 + t < K) f[(size_t)(i0 + t) * M1 + m] = acc[t];
}

}  // namespace bte
