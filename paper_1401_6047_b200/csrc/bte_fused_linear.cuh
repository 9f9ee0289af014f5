// bte_fused_linear.cuh -- the production step kernel of libbte_b200 (sm_100a).
//
// One launch = one leap-frog step (eq. 40-41) of every active system: whole-grid update, fractional-grid
// update, norm / drift-velocity reductions and the running sums of eq. (17), 64 B of HBM traffic per
// lattice point (each of a_h, b_h, a_f, b_f read once and written once, ping-pong buffers).
//
// Work decomposition ("linearised static partition"): the lattice of every active system is cut into
// strips of W = T-2 phi_y columns; the row-units (system, strip, row n) are numbered consecutively and
// dealt out in equal contiguous ranges to a persistent grid of one wave of CTAs (grid = SMs x resident
// CTAs).  A CTA walks its range as one or more segments (system, strip, rows r0 .. r0+Lr-1); within a
// segment it marches over n, every row staged once through an 8-slot shared-memory ring by cp.async, so
// the only redundant work is the 2-row / 2-column halo of a segment.  Rows outside [0, N] are the zero
// ghost rows of the layout (bte_device.cuh), columns outside [0, M] are zero-filled by cp.async: the
// boundary conditions (22)-(23) need no branch in the steady-state iteration.
//
// Iteration u of a segment (arriving row ra = r0-2+u), one __syncthreads:
//   dF(ra)        = F_old[ra][m+1] - F_old[ra][m-1]
//   H_new[ra-1]   from H_old[ra-1], dF(ra-2), dF(ra)           -> global, 2-slot smem ring   (eq. 40)
//   dH(ra-2)      from the ring row written one iteration ago
//   F_new[ra-3]   from F_old[ra-3], dH(ra-4), dH(ra-2)         -> global                     (eq. 41, C5)
// The body exists twice: EDGE = true (first 6 and last 6 iterations of a segment: special rows 0 and 1,
// halo rows, partial prefetch) and EDGE = false (steady state, no row predicates).
#pragma once
#include <type_traits>

#include "bte_kernels.cuh"

namespace bte {

template <int T>
struct LinCfg {
    static constexpr int D = 3;            // rows prefetched ahead of the arriving row
    static constexpr int R = 8;            // ring slots: units u-3..u live, u+1..u+D+1 in flight  (D+5)
    static constexpr int W = T - 2;
    static constexpr int FCOLS = T + 2;
    static constexpr int MAX_SPAN = 64;    // distinct systems one CTA range may touch
    static constexpr size_t smem_bytes = sizeof(double2) * ((size_t)R * (FCOLS + T) + 2 * T);
};

__device__ __forceinline__ bool sys_active(const Layout& L, int s) {
    const long long tot = L.sc[s].n_steps_total;
    return tot == 0 || L.ss[s].k < tot;
}

__device__ __forceinline__ void cp_async16_sz(unsigned smem_addr, const void* gmem_src, int src_bytes) {
    asm volatile("cp.async.cg.shared.global [%0], [%1], 16, %2;\n" ::"r"(smem_addr), "l"(gmem_src),
                 "r"(src_bytes)
                 : "memory");
}
__device__ __forceinline__ void cp_async16_sz_if(unsigned smem_addr, const void* gmem_src, int src_bytes,
                                                 int pred) {
    asm volatile(
        "{\n .reg .pred p;\n setp.ne.s32 p, %3, 0;\n"
        " @p cp.async.cg.shared.global [%0], [%1], 16, %2;\n}\n" ::"r"(smem_addr),
        "l"(gmem_src), "r"(src_bytes), "r"(pred)
        : "memory");
}
__device__ __forceinline__ double2 lds_d2(unsigned addr) {
    double2 v;
    asm volatile("ld.shared.v2.f64 {%0, %1}, [%2];\n" : "=d"(v.x), "=d"(v.y) : "r"(addr));
    return v;
}
__device__ __forceinline__ void sts_d2(unsigned addr, double2 v) {
    asm volatile("st.shared.v2.f64 [%0], {%1, %2};\n" ::"r"(addr), "d"(v.x), "d"(v.y) : "memory");
}

// One segment: system sys, strip, rows r0 .. r0+Lr-1.
template <int T>
__device__ __forceinline__ void linear_segment(const Layout& L, const int sys, const int strip, const int r0,
                                               const int Lr, const int n_strips, const unsigned ups,
                                               double2* smem, double* Es, double* red, double (*s_acc)[T],
                                               unsigned int* s_flag) {
    using Cfg = LinCfg<T>;
    constexpr int D = Cfg::D, R = Cfg::R, W = Cfg::W, FCOLS = Cfg::FCOLS;
    constexpr unsigned FROW = FCOLS * 16, HROW = T * 16;   // ring row strides in bytes
    const int i = threadIdx.x;
    const unsigned sF = (unsigned)__cvta_generic_to_shared(smem);          // F ring  [R][FCOLS]
    const unsigned sH = sF + R * FROW;                                      // H ring  [R][T]
    const unsigned sN = sH + R * HROW;                                      // Hn ring [2][T]

    const SysConst c = L.sc[sys];
    const long long k = L.ss[sys].k;
    const int cur = (int)(k & 1), nxt = cur ^ 1;
    // one input and one output base pointer; the fractional grid of the same buffer sits Y elements
    // further (Y = n_batch * points per array < 2^30, checked by the host), folded into 32-bit offsets
    const double2* __restrict__ Hold = state_ptr(L, cur, 0, sys);
    double2* __restrict__ Hnew = state_ptr(L, nxt, 0, sys);
    const int Y = L.n_batch * (L.N + 1 + 2 * GHOST) * L.pitch;
    int cn_idx = sys * (L.N + 1 + 2 * GHOST) + GHOST;     // index of c_0 of this system in L.cn

    const int c0 = strip * W;
    const int col = c0 - 1 + i;
    const bool col_valid = (col >= 0) && (col < L.M1);
    const bool owner = (i >= 1) && (i <= W) && col_valid;
    const int cf = c0 - 2 + i;                         // this thread's F_old column in the ring
    const int szF = (cf >= 0 && cf < L.M1) ? 16 : 0;   // cp.async src sizes: 0 => zero fill (eq. 22-23 in m)
    const int cf2 = c0 - 2 + T + i;                    // threads 0, 1: the two extra columns
    const int szF2 = (cf2 < L.M1) ? 16 : 0;
    const int szH = col_valid ? 16 : 0;
    const int ipitch = L.pitch;
    const int adjH = col_valid ? col : 0;
    const int adjF = (szF ? cf : 0) + Y, adjF2 = ((i < 2 && szF2) ? cf2 : 0) + Y;
    const int two = (i < 2) ? 1 : 0;

    __syncthreads();   // the previous segment (or the scan) is done with Es / rings / red / s_acc
    if (i < 4) Es[i] = field_E(c, ((double)k + 0.5 * (double)i) * L.dt);   // t_k .. t_{k+3/2} (C14)
    const double2 zero = make_double2(0.0, 0.0);
    sts_d2(sN + i * 16, zero);
    sts_d2(sN + HROW + i * 16, zero);
    s_acc[0][i] = 0.0;
    s_acc[1][i] = 0.0;

    const int u_start = (r0 == 0) ? 2 : 0;             // rows -2, -1 are zero: skip their iterations
    const int n_iter = Lr + 5;
    const int h_lo = max(0, r0 - 1), h_hi = min(L.N, r0 + Lr);   // whole-grid rows formed in this segment

    // issue of load unit v (F_old row r0-2+v, H_old row r0-2+v) into ring slot v & 7
    int off_in = (r0 - 2 + u_start) * ipitch;          // element offset of the next unit's row
    auto issue_edge = [&](int v) {
        if (v <= Lr + 3) {
            const unsigned slot = (unsigned)(v & (R - 1));
            cp_async16_sz(sF + slot * FROW + i * 16, Hold + (off_in + adjF), szF);
            cp_async16_sz_if(sF + slot * FROW + (T + i) * 16, Hold + (off_in + adjF2), szF2, two);
            if (v >= 1 && v <= Lr + 2) cp_async16_sz(sH + slot * HROW + i * 16, Hold + (off_in + adjH), szH);
        }
        cp_async_commit();
        off_in += ipitch;
    };
#pragma unroll
    for (int v = 0; v <= D; ++v) issue_edge(u_start + v);

    const double ph = col_valid ? L.phi[(size_t)sys * L.pitch + col] : 0.0;
    const double gdt = col_valid ? __dmul_rn(L.gm[(size_t)sys * L.pitch + col], L.dt) : 0.0;
    const double kappa = col_valid ? c.kappa_dt : 0.0;   // invalid columns: w = 0, src = 0, kappa = 0 => 0
    __syncthreads();   // Es visible
    const double hbHa = __dmul_rn(__fma_rn(c.B, ph, Es[0]), L.hd);   // whole grid: explicit time t_k
    const double hbHb = __dmul_rn(__fma_rn(c.B, ph, Es[2]), L.hd);   //             implicit time t_{k+1}
    const double hbFa = __dmul_rn(__fma_rn(c.B, ph, Es[1]), L.hd);   // fractional grid: t_{k+1/2}
    const double hbFb = __dmul_rn(__fma_rn(c.B, ph, Es[3]), L.hd);   //                  t_{k+3/2}

    double2 dF1 = zero, dF2 = zero, dH1 = zero, dH2 = zero;
    int jH = r0 - 3 + u_start;                          // whole-grid row of the current iteration
    auto load_cn = [&](int j) { return (j >= -GHOST && j <= L.N + GHOST) ? __ldg(L.cn + (cn_idx + j)) : 0.0; };
    double cF = load_cn(jH - 2), cM = load_cn(jH - 1);
    int cn_j = cn_idx + jH;                              // index of c_{jH}
    double ndH = (double)jH;
    int off_out = jH * ipitch + adjH;                   // element offset of (jH, col)
    const int dFo = Y - 2 * ipitch;                     // (jH, col) of H_new -> (jH-2, col) of F_new
    const unsigned tF = sF + i * 16;
    constexpr unsigned tH_off = R * FROW, tN_off = R * FROW + R * HROW;   // H ring, Hn ring relative to tF

    auto body = [&](auto edge_tag, const int u) {
        constexpr bool EDGE = decltype(edge_tag)::value;
        const unsigned su = (unsigned)(u & (R - 1));
        const unsigned o_u = su * FROW;                              // unit u  : arriving F_old row
        const unsigned o_f = ((su + 5) & (R - 1)) * FROW;           // unit u-3: F_old row jF
        const unsigned o_h = ((su + 7) & (R - 1)) * HROW;           // unit u-1: H_old row jH
        const unsigned si = (su + D + 1) & (R - 1);                  // unit u+D+1 (slot of dead unit u-4)
        const unsigned nw = (unsigned)(u & 1) * HROW, nr = HROW - nw;   // Hn ring: write / read slot

        cp_async_wait<D>();   // this thread's copies of unit u have landed
        __syncthreads();      // ... everybody's; orders the Hn ring; frees slot (u-4) & 7
        const double cH = EDGE ? load_cn(jH) : __ldg(L.cn + cn_j);
        if (EDGE) {
            issue_edge(u + D + 1);
        } else {
            cp_async16_sz(tF + si * FROW, Hold + (off_in + adjF), szF);
            cp_async16_sz_if(tF + si * FROW + T * 16, Hold + (off_in + adjF2), szF2, two);
            cp_async16_sz(tF + tH_off + si * HROW, Hold + (off_in + adjH), szH);
            cp_async_commit();
            off_in += ipitch;
        }
        // dF of the arriving row (row 0 pre-doubled in a: chi(1) = 2, eq. 11)
        double2 dF0;
        {
            const double2 l = lds_d2(tF + o_u), r = lds_d2(tF + o_u + 32);
            dF0.x = __dsub_rn(r.x, l.x); dF0.y = __dsub_rn(r.y, l.y);
            if (EDGE && jH + 1 == 0) dF0.x *= 2.0;
        }
        // whole grid, row jH (eq. 40)
        double2 hn = zero;
        if (!EDGE || (jH >= h_lo && jH <= h_hi)) {
            const double2 w = lds_d2(tF + tH_off + o_h);
            hn = cn_point(w, dF2, dF0, ndH, hbHa, hbHb, __dmul_rn(cH, gdt), kappa, L.xi, L.nu, L.nu2);
            if (EDGE) {
                if (jH == 0) hn.y = 0.0;   // b_0 == 0 (eq. 23, C3)
                if (owner && jH >= r0 && jH < r0 + Lr) {
                    Hnew[off_out] = hn;
                    if (jH == 0) s_acc[0][i] = hn.x;
                    if (jH == 1) {
                        s_acc[1][i] = hn.y;
                        if (col == 0) L.ss[sys].edge[0] = fabs(hn.y);
                        if (col == L.M1 - 1) L.ss[sys].edge[1] = fabs(hn.y);
                    }
                }
            } else {
                if (owner) Hnew[off_out] = hn;
            }
        }
        sts_d2(tF + tN_off + nw, hn);
        // dH of row jH-1, written one iteration ago (visible since this iteration's barrier)
        double2 dH0 = zero;
        if (i >= 1 && i <= W) {
            const double2 l = lds_d2(tF + tN_off + nr - 16), r = lds_d2(tF + tN_off + nr + 16);
            dH0.x = __dsub_rn(r.x, l.x); dH0.y = __dsub_rn(r.y, l.y);
            if (EDGE && jH - 1 == 0) dH0.x *= 2.0;
        }
        // fractional grid, row jF = jH-2 (eq. 41): stencil from the NEW whole grid (C5)
        if (EDGE) {
            const int jF = jH - 2;
            if (owner && jF >= r0 && jF < r0 + Lr) {
                const double2 w = lds_d2(tF + o_f + 16);
                double2 fn = cn_point(w, dH2, dH0, ndH - 2.0, hbFa, hbFb, __dmul_rn(cF, gdt), kappa, L.xi,
                                      L.nu, L.nu2);
                if (jF == 0) fn.y = 0.0;
                Hnew[off_out + dFo] = fn;
            }
        } else {
            const double2 w = lds_d2(tF + o_f + 16);
            const double2 fn = cn_point(w, dH2, dH0, ndH - 2.0, hbFa, hbFb, __dmul_rn(cF, gdt), kappa, L.xi,
                                        L.nu, L.nu2);
            if (owner) Hnew[off_out + dFo] = fn;
        }
        dF2 = dF1; dF1 = dF0;
        dH2 = dH1; dH1 = dH0;
        cF = cM; cM = cH;
        ++jH; ++cn_j; ndH += 1.0;
        off_out += ipitch;
    };

    // steady state: u in [6, Lr-2] (all of ra, jH, jF are interior rows of the segment, prefetch in range)
    const int u_steady_end = Lr - 2;
    int u = u_start;
    for (; u < min(6, n_iter); ++u) body(std::true_type{}, u);
#pragma unroll 3
    for (; u <= u_steady_end; ++u) body(std::false_type{}, u);
    for (; u < n_iter; ++u) body(std::true_type{}, u);
    cp_async_wait<0>();

    // per-strip partial sums of row 0 (a) and row 1 (b) -> eq. (12), (20)
    const bool has0 = (r0 == 0), has1 = (r0 <= 1) && (r0 + Lr > 1);
    double* part = L.partial + ((size_t)sys * L.pitch + strip) * 2;
    if (has0) {
        const double s = warp_sum(s_acc[0][i]);
        if ((i & 31) == 0) red[i >> 5] = s;
        __syncthreads();
        if (i == 0) {
            double t = 0.0;
#pragma unroll
            for (int w = 0; w < T / 32; ++w) t += red[w];
            part[0] = t;
        }
        __syncthreads();
    }
    if (has1) {
        const double s = warp_sum(s_acc[1][i]);
        if ((i & 31) == 0) red[i >> 5] = s;
        __syncthreads();
        if (i == 0) {
            double t = 0.0;
#pragma unroll
            for (int w = 0; w < T / 32; ++w) t += red[w];
            part[1] = t;
        }
    }
    // the CTA that completes the last row-unit of this system folds its partial sums (k unchanged)
    __threadfence();
    __syncthreads();
    if (i == 0) {
        const unsigned int prev = atomicAdd(&L.ss[sys].done, (unsigned int)Lr);
        *s_flag = (prev + (unsigned int)Lr == ups) ? 1u : 0u;
    }
    __syncthreads();
    if (*s_flag && i < 32) {
        __threadfence();
        fold_and_advance(L, sys, n_strips, k, 2);
    }
}

// BUDGETS: some system has a step budget (n_steps_total > 0) => the active set is compacted on the fly.
template <int T, bool BUDGETS, int MINB>
__global__ void __launch_bounds__(T, MINB) fused_linear_kernel(const __grid_constant__ Layout L) {
    using Cfg = LinCfg<T>;
    constexpr int W = Cfg::W;
    static_assert(Cfg::D + 5 == Cfg::R && (Cfg::R & (Cfg::R - 1)) == 0, "ring size");
    extern __shared__ double2 smem[];
    __shared__ double Es[4];
    __shared__ double red[T / 32];
    __shared__ double s_acc[2][T];   // row 0 (a) and row 1 (b) of the new whole grid, per owned column
    __shared__ int s_scan[T / 32];
    __shared__ int s_list[Cfg::MAX_SPAN];
    __shared__ unsigned int s_flag;

    const int i = threadIdx.x;
    const int rows = L.N + 1;
    const int n_strips = (L.M1 + W - 1) / W;
    const unsigned ups = (unsigned)n_strips * (unsigned)rows;     // row-units per system (< 2^31)

    // ---- active systems and this CTA's range of row-units -------------------------------------------
    long long n_active = L.n_batch;
    int a_first = 0;
    long long start, end;
    if (BUDGETS) {
        const int q = (L.n_batch + T - 1) / T;            // systems scanned per thread
        const int s_lo = min(i * q, L.n_batch), s_hi = min(s_lo + q, L.n_batch);
        int cnt = 0;
        for (int s = s_lo; s < s_hi; ++s) cnt += sys_active(L, s) ? 1 : 0;
        int incl = cnt;                                   // inclusive scan over the CTA
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) {
            const int v = __shfl_up_sync(0xffffffffu, incl, o);
            if ((i & 31) >= o) incl += v;
        }
        if ((i & 31) == 31) s_scan[i >> 5] = incl;
        __syncthreads();
        int base = 0, total = 0;
#pragma unroll
        for (int w = 0; w < T / 32; ++w) {
            if (w < (i >> 5)) base += s_scan[w];
            total += s_scan[w];
        }
        n_active = total;
        const long long units = n_active * ups;
        const long long U = (units + gridDim.x - 1) / gridDim.x;
        start = min((long long)blockIdx.x * U, units);
        end = min(start + U, units);
        if (start < end) {
            a_first = (int)(start / ups);
            const int a_last = (int)((end - 1) / ups);
            int a = base + incl - cnt;                    // index of this thread's first active system
            for (int s = s_lo; s < s_hi; ++s) {
                if (sys_active(L, s)) {
                    if (a >= a_first && a <= a_last) s_list[a - a_first] = s;
                    ++a;
                }
            }
        }
        __syncthreads();
    } else {
        const long long units = n_active * ups;
        const long long U = (units + gridDim.x - 1) / gridDim.x;
        start = min((long long)blockIdx.x * U, units);
        end = min(start + U, units);
    }

    // ---- walk the range segment by segment -----------------------------------------------------------
    long long pos = start;
    while (pos < end) {
        const int a = (int)(pos / ups);
        const int rem = (int)(pos - (long long)a * ups);
        const int strip = rem / rows;
        const int r0 = rem - strip * rows;
        const int Lr = (int)min((long long)(rows - r0), end - pos);
        const int sys = BUDGETS ? s_list[a - a_first] : a;
        pos += Lr;
        linear_segment<T>(L, sys, strip, r0, Lr, n_strips, ups, smem, Es, red, s_acc, &s_flag);
    }

    // ---- the last CTA of the launch advances the step counters of all systems that were active --------
    __threadfence();
    __syncthreads();
    if (i == 0) {
        const unsigned int prev = atomicAdd(L.gctl, 1u);
        s_flag = (prev + 1u == gridDim.x) ? 1u : 0u;
    }
    __syncthreads();
    if (s_flag) {
        __threadfence();
        for (int s = i; s < L.n_batch; s += T)
            if (sys_active(L, s)) L.ss[s].k += 1;
        if (i == 0) *L.gctl = 0u;
    }
}

}  // namespace bte
