// bte_sweep.cuh -- the production step kernel of libbte_b200 (sm_100a): S leap-frog steps per sweep.
//
// One launch = S consecutive leap-frog steps (eq. 40-41) of every active system = NS = 2 S applications of
// T (eq. 38), alternating whole grid / fractional grid, in ONE pass over the lattice: each of a_h, b_h,
// a_f, b_f is read once and written once per launch (ping-pong buffers), i.e. 64/S bytes of HBM traffic per
// lattice point per time step.  S = 1 is the plain fused whole+fractional step; S >= 2 is temporal
// blocking: the intermediate time levels live only in shared-memory rings.  The per-step reductions
// (norm eq. 12, drift velocity eq. 20, running sums of eq. 17) are produced for every one of the S steps.
//
// Work decomposition ("linearised static partition"): the lattice of every active system is cut into
// strips of W = T - 2 (NS-1) phi_y columns (the other 2 (NS-1) threads of a CTA recompute halo columns);
// the row-units (system, strip, row n) are numbered consecutively and dealt out in equal contiguous ranges
// to a persistent grid of one wave of CTAs.  A CTA walks its range as segments (system, strip, rows
// r0 .. r0+Lr-1) and marches over n inside a segment.
//
// Pipeline of a segment.  Iteration u: row ra = r0 - NS + u of F^0 (the fractional grid in HBM) and row
// ra - 1 of H^0 (whole grid) have arrived in an 8-slot shared-memory ring (cp.async, 3 rows ahead; columns
// outside [0, M] and rows outside [0, N] are zero-filled = boundary conditions (22)-(23)).  Stage j = 0 .. NS-1 forms row  row_j = ra - 1 - 2 j  of time level j+1:
//     X^{j+1}[row_j] = T( own = X^{j-1}[row_j] ; stencil rows row_j -+ 1 of X^j )
// (even j: whole grid, odd j: fractional grid; X^0 = F^0, X^{-1} = H^0).  Stage j writes its row into a
// shared-memory ring; one iteration (= one __syncthreads) later stage j+1 takes the phi_y-difference of that
// row, and four iterations later stage j+2 reads it back as its own point.  The last whole-grid stage and the
// last fractional stage also store to HBM.  One barrier per iteration, no other synchronisation.
// The body exists twice: EDGE = true (pipeline fill / drain of a segment: special rows 0 and 1, halo rows,
// partial prefetch) and EDGE = false (steady state, no row predicates).
#pragma once
#include <type_traits>

#include "bte_kernels.cuh"

namespace bte {

template <int T, int S>
struct SweepCfg {
    static constexpr int NS = 2 * S;           // half-updates (stages) per sweep
    static constexpr int HALO = NS - 1;        // halo columns on each side of a strip, halo rows of a segment
    static constexpr int W = T - 2 * HALO;     // owned columns per strip
    static constexpr int D = 3;                // rows prefetched ahead of the arriving row
    static constexpr int R = 8;                // input ring slots: units u-3..u live, u+1..u+D+1 in flight
    static constexpr int FCOLS = T + 2;        // F^0 columns per ring row
    static constexpr int SC = T + 2;           // stage ring row: T columns + one zero pad column each side
    static constexpr int QD = 8;               // depth of a stage ring that is read back as "own" (4 iterations later)
    static constexpr int ring_rows = (NS - 2) * QD + 2;   // stages 0..NS-3: QD slots; stage NS-2: 2 slots
    static constexpr int MAX_SPAN = 64;        // distinct systems one CTA range may touch
    static constexpr int CS = 32;              // c_n ring: unit v brings c of its row into slots v & 15 and (v & 15) + 16
    static constexpr size_t smem_bytes = sizeof(double2) * ((size_t)R * (FCOLS + T) + (size_t)ring_rows * SC) + CS * sizeof(double);
    static_assert(W >= 32, "strip too narrow");
    static_assert(2 * (NS - 1) + 1 + D + 1 <= 16, "c_n ring too short");
};

// active for an S-step launch: no budget, or at least S steps left (the host never issues an S-step launch
// while a system has fewer than S but more than 0 steps left, bte.cu)
__device__ __forceinline__ bool sys_active(const Layout& L, int s, int S) {
    const long long tot = L.sc[s].n_steps_total;
    return (tot == 0 || L.ss[s].k + S <= tot) && L.ss[s].phase != 2;   // (phase 2: finished by the steady-state policy)
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
// 8-byte copy issued by thread 0 only (c_n of the row of a load unit); src_bytes 0 => zero fill
__device__ __forceinline__ void cp_async8_sz_if(unsigned smem_addr, const void* gmem_src, int src_bytes,
                                                int pred) {
    asm volatile(
        "{\n .reg .pred p;\n setp.ne.s32 p, %3, 0;\n"
        " @p cp.async.ca.shared.global [%0], [%1], 8, %2;\n}\n" ::"r"(smem_addr),
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
__device__ __forceinline__ double lds_d(unsigned addr) {
    double v;
    asm volatile("ld.shared.f64 %0, [%1];\n" : "=d"(v) : "r"(addr));
    return v;
}

// Fold of the per-strip partial sums of the S steps of one sweep and the per-step bookkeeping of one
// system, executed by warp 0 of the CTA that completed the system's last row-unit (fixed summation order
// => deterministic).  eq. (12), (20) by the rectangle rule (C10); running sums of eq. (17) for steps
// k+s+1 > avg_start (C9).  The step counter itself is advanced by the last CTA of the launch.
__device__ __forceinline__ void fold_sweep(const Layout& L, int sys, int n_partials, long long k, int S) {
    const int lane = threadIdx.x & 31;
    const SysConst c = L.sc[sys];
    SysState* st = L.ss + sys;
    for (int s = 0; s < S; ++s) {
        // (the fold of the last system is the very end of a launch: the partial sums are read from L2 with independent
        // 128-bit loads, several in flight, not one dependent round trip per value)
        const double2* part = (const double2*)(L.partial + ((size_t)s * L.n_batch + sys) * L.pitch * 2);
        double sa = 0.0, sb = 0.0;
#pragma unroll 4
        for (int p = lane; p < n_partials; p += 32) {
            const double2 v = __ldcg(part + p);
            sa += v.x;
            sb += v.y;
        }
        sa = warp_sum(sa);
        sb = warp_sum(sb);
        if (lane == 0) {
            const double norm = c.norm_scale * sa;
            const double v = c.v_scale * sb;
            st->norm = norm;
            st->v_dr = v;
            accumulate_step(c, st, v, k + s + 1, L.dt);
        }
    }
    if (lane == 0) {
        st->edge_leak = ((volatile double*)st->edge)[0] + ((volatile double*)st->edge)[1];
        st->done = 0u;
        __threadfence();
    }
}

// Static shared memory of the sweep kernel.
template <int T, int S>
struct SweepShared {
    double Es[2 * S + 2];            // E(t_k + v dt/2), v = 0 .. NS+1  (C14)
    double red[T / 32];
    double acc[S][2][T];             // rows 0 (a) and 1 (b) of the S new whole grids, per owned column
    int scan[T / 32];
    int list[SweepCfg<T, S>::MAX_SPAN];
    unsigned int flag;
};

// One segment: system sys, strip, rows r0 .. r0+Lr-1.
// SKIP: in the fill / drain iterations do not compute stages whose row lies outside their range (a uniform branch);
// pays off for batches of short columns, where fill / drain is a large share of a segment (used when BUDGETS).
template <int T, int S, bool SKIP>
__device__ __forceinline__ void sweep_segment(const Layout& L, const int sys, const int strip, const int r0,
                                              const int Lr, const int n_strips, const unsigned ups,
                                              double2* smem, SweepShared<T, S>& sh) {
    using Cfg = SweepCfg<T, S>;
    constexpr int NS = Cfg::NS, HALO = Cfg::HALO, D = Cfg::D, R = Cfg::R, W = Cfg::W, FCOLS = Cfg::FCOLS;
    constexpr int SC = Cfg::SC, QD = Cfg::QD;
    constexpr unsigned FROW = FCOLS * 16, HROW = T * 16, SROW = SC * 16;   // ring row strides in bytes
    const int i = threadIdx.x;
    const unsigned sF = (unsigned)__cvta_generic_to_shared(smem);          // F^0 ring [R][FCOLS]
    const unsigned sH = sF + R * FROW;                                      // H^0 ring [R][T]
    const unsigned sC = sH + R * HROW + Cfg::ring_rows * SROW;             // c_n ring [CS] doubles

    const SysConst c = L.sc[sys];
    const long long k = L.ss[sys].k;
    const int cur = L.ss[sys].buf, nxt = cur ^ 1;
    // one input and one output base pointer; the fractional grid of the same buffer sits Y elements
    // further (Y = n_batch * points per array < 2^30, checked by the host), folded into 32-bit offsets
    const double2* __restrict__ Hold = state_ptr(L, cur, 0, sys);
    double2* __restrict__ Hnew = state_ptr(L, nxt, 0, sys);
    const int Y = L.n_batch * (L.N + 1 + 2 * GHOST) * L.pitch;
    const double* __restrict__ cn0 = cn_ptr(L, sys);      // c_0 of this system

    const int c0 = strip * W;
    const int col = c0 - HALO + i;
    const bool col_valid = (col >= 0) && (col < L.M1);
    const bool owner = (i >= HALO) && (i < HALO + W) && col_valid;
    const int cf = col - 1;                            // this thread's F^0 column in the ring
    const int szF = (cf >= 0 && cf < L.M1) ? 16 : 0;   // cp.async src sizes: 0 => zero fill (eq. 22-23 in m)
    const int cf2 = cf + T;                            // threads 0, 1: the two extra columns
    const int szF2 = (cf2 >= 0 && cf2 < L.M1) ? 16 : 0;
    const int szH = col_valid ? 16 : 0;
    const int ipitch = L.pitch;
    const int adjH = col_valid ? col : 0;
    const int adjF = (szF ? cf : 0) + Y, adjF2 = ((i < 2 && szF2) ? cf2 : 0) + Y;
    const int two = (i < 2) ? 1 : 0;

    __syncthreads();   // the previous segment (or the scan) is done with the rings / sh
    if (i < NS + 2) sh.Es[i] = field_E(c, ((double)k + 0.5 * (double)i) * L.dt);   // (C14)
#pragma unroll
    for (int s = 0; s < S; ++s) {
        sh.acc[s][0][i] = 0.0;
        sh.acc[s][1][i] = 0.0;
    }

    const int u_start = (r0 == 0) ? NS : 0;            // rows -NS .. -1 are zero: skip their iterations
    const int n_iter = Lr + 3 * NS - 1;
    const int row_first = r0 - NS - 1;                 // stage 0's row at iteration u is row_first + u

    // issue of load unit v (F^0 row r0-NS+v, H^0 row r0-NS+v) into ring slot v & 7
    int off_in = (r0 - NS + u_start) * ipitch;         // element offset of the next unit's row
    auto issue_edge = [&](int v) {
        if (v <= Lr + 2 * NS - 1) {
            const unsigned slot = (unsigned)(v & (R - 1));
            const int row = r0 - NS + v;
            const bool in = (row >= 0) && (row <= L.N);   // rows outside the lattice: zero fill, nothing read
            const int o = in ? off_in : 0;
            cp_async16_sz(sF + slot * FROW + i * 16, Hold + (o + adjF), in ? szF : 0);
            cp_async16_sz_if(sF + slot * FROW + (T + i) * 16, Hold + (o + adjF2), in ? szF2 : 0, two);
            if (v >= 1 && v <= Lr + 2 * NS - 2) cp_async16_sz(sH + slot * HROW + i * 16, Hold + (o + adjH), in ? szH : 0);
            cp_async8_sz_if(sC + (unsigned)((v & 15) + 16 * i) * 8, cn0 + (in ? row : 0), in ? 8 : 0, two);
        }
        cp_async_commit();
        off_in += ipitch;
    };
#pragma unroll
    for (int v = 0; v <= D; ++v) issue_edge(u_start + v);

    const double ph = col_valid ? L.phi[(size_t)sys * L.pitch + col] : 0.0;
    const double gdt = col_valid ? __dmul_rn(L.gm[(size_t)sys * L.pitch + col], L.dt) : 0.0;
    const double kappa = col_valid ? c.kappa_dt : 0.0;   // invalid columns: w = 0, src = 0, kappa = 0 => 0
    __syncthreads();   // Es, cs visible
    double hb[NS + 2];                                   // beta^t_m dt/2 at the NS+2 half-step times (eq. 28-29)
#pragma unroll
    for (int v = 0; v < NS + 2; ++v) hb[v] = __dmul_rn(__fma_rn(c.B, ph, sh.Es[v]), L.hd);

    const double2 zero = make_double2(0.0, 0.0);
    double2 d1[NS], d2[NS];                              // phi_y-differences formed 1 and 2 iterations ago
#pragma unroll
    for (int j = 0; j < NS; ++j) d1[j] = d2[j] = zero;

    int row0 = row_first + u_start;                     // stage 0's row in the current iteration
    double nd0 = (double)row0;
    int off_out = (row0 - 2 * (NS - 2)) * ipitch + adjH;   // element offset of (row of stage NS-2, col) in H_new
    const int dFo = Y - 2 * ipitch;                     // ... -> (row of stage NS-1, col) of F_new
    const unsigned tF = sF + i * 16;
    constexpr unsigned tH_off = R * FROW, tQ_off = R * FROW + R * HROW;   // H ring, stage rings relative to tF

    // slot_tag: std::integral_constant<int, K>: K = u & 7 known at compile time (all ring offsets become
    // immediates), or K = -1: taken from u at run time
    auto body = [&](auto edge_tag, auto slot_tag, const int u) {
        constexpr bool EDGE = decltype(edge_tag)::value;
        constexpr int K = decltype(slot_tag)::value;
        const unsigned su = K >= 0 ? (unsigned)K : (unsigned)(u & (R - 1));
        const unsigned o_u = su * FROW;                              // unit u  : arriving F^0 row
        const unsigned o_f = ((su + 5) & (R - 1)) * FROW;           // unit u-3: F^0 row of stage 1
        const unsigned o_h = ((su + 7) & (R - 1)) * HROW;           // unit u-1: H^0 row of stage 0
        const unsigned si = (su + D + 1) & (R - 1);                  // unit u+D+1 (slot of dead unit u-4)
        const unsigned q_w = su * SROW;                              // stage ring (depth 8): slot written now
        const unsigned q_p = ((su + 7) & (R - 1)) * SROW;           //   slot written one iteration ago
        const unsigned q_o = ((su + 4) & (R - 1)) * SROW;           //   slot written four iterations ago
        const unsigned l_w = (su & 1u) * SROW, l_p = SROW - l_w;      // last stage ring (depth 2)
        // c_n ring: unit v sits in slots v & 15 and (v & 15) + 16, so that unit u-1 and the NS-1 older ones
        // (2 apart) are read at descending addresses from one base without wrap-around
        const unsigned c_b = sC + (((su + 7) & (R - 1)) + ((unsigned)(u - 1) & 8u) + 16u) * 8;
        static_assert(QD == R, "stage ring slots share the input ring's slot arithmetic");

        cp_async_wait<D>();   // this thread's copies of unit u have landed
        __syncthreads();      // ... everybody's; orders the stage rings; frees slot (u-4) & 7
        if (EDGE) {
            issue_edge(u + D + 1);
        } else {
            cp_async16_sz(tF + si * FROW, Hold + (off_in + adjF), szF);
            cp_async16_sz_if(tF + si * FROW + T * 16, Hold + (off_in + adjF2), szF2, two);
            cp_async16_sz(tF + tH_off + si * HROW, Hold + (off_in + adjH), szH);
            cp_async8_sz_if(sC + (((su + D + 1) & (R - 1)) + ((unsigned)(u + D + 1) & 8u) + 16u * i) * 8,
                            cn0 + (row0 + D + 2), 8, two);
            cp_async_commit();
            off_in += ipitch;
        }
        // phase 1: every shared-memory read of this iteration (all of them target slots written in earlier
        // iterations, so they are independent of this iteration's results and can be in flight together)
        double2 d0s[NS], ws[NS];
        double cjs[NS];
        bool act[NS];
#pragma unroll
        for (int j = 0; j < NS; ++j) {
            const int row = row0 - 2 * j;                            // row formed by stage j
            act[j] = true;
            if (EDGE && SKIP) { ws[j] = zero; cjs[j] = 0.0; }
            // phi_y-difference of row+1 of the stencil grid X^j (row 0 pre-doubled in a: chi(1) = 2, eq. 11)
            {
                unsigned a;
                if (j == 0) a = tF + o_u;                                        // F^0, columns col-1 / col+1
                else if (j == NS - 1) a = tF + tQ_off + (NS - 2) * QD * SROW + l_p;
                else a = tF + tQ_off + (j - 1) * QD * SROW + q_p;
                const double2 l = lds_d2(a), r = lds_d2(a + 32);
                d0s[j].x = __dsub_rn(r.x, l.x); d0s[j].y = __dsub_rn(r.y, l.y);
                if (EDGE && row + 1 == 0) d0s[j].x *= 2.0;
            }
            if (EDGE && SKIP) {
                act[j] = row >= max(0, r0 - (HALO - j)) && row <= min(L.N, r0 + Lr - 1 + (HALO - j));
                if (!act[j]) continue;                               // uniform over the CTA
            }
            // own point: X^{j-1}[row][col]
            if (j == 0) ws[j] = lds_d2(tF + tH_off + o_h);
            else if (j == 1) ws[j] = lds_d2(tF + o_f + 16);
            else ws[j] = lds_d2(tF + tQ_off + (j - 2) * QD * SROW + q_o + 16);
            cjs[j] = lds_d(c_b - 16 * j);                             // unit u-1-2j brought c of this row
        }
        // phase 2: the NS half-updates
#pragma unroll
        for (int j = 0; j < NS; ++j) {
            const int row = row0 - 2 * j;
            const double2 d0 = d0s[j], w = ws[j];
            const double cj = cjs[j];
            double2 out = zero;
            if (!(EDGE && SKIP) || act[j]) {
                out = cn_point(w, d2[j], d0, nd0 - (double)(2 * j), hb[j], hb[j + 2], __dmul_rn(cj, gdt), kappa, L.xi,
                               L.nu, L.nu2);
                if (EDGE) {
                    const int lo = max(0, r0 - (HALO - j)), hi = min(L.N, r0 + Lr - 1 + (HALO - j));
                    if (row < lo || row > hi) out = zero;    // outside the lattice / outside this segment's halo
                    if (row == 0) out.y = 0.0;               // b_0 == 0 (eq. 23, C3)
                }
            }
            if (j < NS - 2) sts_d2(tF + tQ_off + j * QD * SROW + q_w + 16, out);
            if (j == NS - 2) sts_d2(tF + tQ_off + (NS - 2) * QD * SROW + l_w + 16, out);
            if (j >= NS - 2) {                            // the two newest time levels go to HBM
                const int o = off_out + (j == NS - 1 ? dFo : 0);
                if (EDGE) {
                    if (owner && row >= r0 && row < r0 + Lr) Hnew[o] = out;
                } else {
                    if (owner) Hnew[o] = out;
                }
            }
            if (EDGE && (j & 1) == 0) {                   // whole grid of step k + j/2 + 1: reductions
                if (owner && row >= r0 && row < r0 + Lr) {
                    if (row == 0) sh.acc[j / 2][0][i] = out.x;
                    if (row == 1) {
                        sh.acc[j / 2][1][i] = out.y;
                        if (j == NS - 2) {
                            if (col == 0) L.ss[sys].edge[0] = fabs(out.y);
                            if (col == L.M1 - 1) L.ss[sys].edge[1] = fabs(out.y);
                        }
                    }
                }
            }
            d2[j] = d1[j]; d1[j] = d0;
        }
        ++row0; nd0 += 1.0;
        off_out += ipitch;
    };

    // steady state: every stage is on an interior row >= 1 of its range, prefetch in range
    // (stage 0 within its rows, the prefetched unit u+D+1 a real row <= N of both input grids)
    const int u_steady_end = min(min(Lr + NS, Lr + 2 * NS - 3 - D), L.N - r0 + NS - D - 1);
    int u = u_start;
    using Dyn = std::integral_constant<int, -1>;
    for (; u < min(3 * NS, n_iter); ++u) body(std::true_type{}, Dyn{}, u);
    while (u <= u_steady_end) {
        if ((u & 7) == 0 && u + 7 <= u_steady_end) {    // 8 iterations with compile-time ring slots
            body(std::false_type{}, std::integral_constant<int, 0>{}, u);
            body(std::false_type{}, std::integral_constant<int, 1>{}, u + 1);
            body(std::false_type{}, std::integral_constant<int, 2>{}, u + 2);
            body(std::false_type{}, std::integral_constant<int, 3>{}, u + 3);
            body(std::false_type{}, std::integral_constant<int, 4>{}, u + 4);
            body(std::false_type{}, std::integral_constant<int, 5>{}, u + 5);
            body(std::false_type{}, std::integral_constant<int, 6>{}, u + 6);
            body(std::false_type{}, std::integral_constant<int, 7>{}, u + 7);
            u += 8;
        } else {
            body(std::false_type{}, Dyn{}, u);
            ++u;
        }
    }
    for (; u < n_iter; ++u) body(std::true_type{}, Dyn{}, u);
    cp_async_wait<0>();

    // per-strip partial sums of row 0 (a) and row 1 (b) of each of the S new whole grids -> eq. (12), (20)
    const bool has0 = (r0 == 0), has1 = (r0 <= 1) && (r0 + Lr > 1);
    if (has0 || has1) {
#pragma unroll
        for (int s = 0; s < S; ++s) {
            double* part = L.partial + (((size_t)s * L.n_batch + sys) * L.pitch + strip) * 2;
#pragma unroll
            for (int q = 0; q < 2; ++q) {
                if (q == 0 ? has0 : has1) {
                    __syncthreads();
                    const double v = warp_sum(sh.acc[s][q][i]);
                    if ((i & 31) == 0) sh.red[i >> 5] = v;
                    __syncthreads();
                    if (i == 0) {
                        double t = 0.0;
#pragma unroll
                        for (int w = 0; w < T / 32; ++w) t += sh.red[w];
                        part[q] = t;
                    }
                }
            }
        }
    }
    // the CTA that completes the last row-unit of this system folds its partial sums (k unchanged)
    __threadfence();
    __syncthreads();
    if (i == 0) {
        const unsigned int prev = atomicAdd(&L.ss[sys].done, (unsigned int)Lr);
        sh.flag = (prev + (unsigned int)Lr == ups) ? 1u : 0u;
    }
    __syncthreads();
    if (sh.flag && i < 32) {
        __threadfence();
        fold_sweep(L, sys, n_strips, k, S);
    }
}

// BUDGETS: some system has a step budget (n_steps_total > 0) => the active set is compacted on the fly.
template <int T, int S, bool BUDGETS, int MINB>
__global__ void __launch_bounds__(T, MINB) sweep_kernel(const __grid_constant__ Layout L) {
    using Cfg = SweepCfg<T, S>;
    constexpr int W = Cfg::W;
    static_assert(Cfg::D + 5 == Cfg::R && (Cfg::R & (Cfg::R - 1)) == 0, "ring size");
    extern __shared__ double2 smem[];
    __shared__ SweepShared<T, S> sh;

    const int i = threadIdx.x;
    const int rows = L.N + 1;
    const int n_strips = (L.M1 + W - 1) / W;
    const unsigned ups = (unsigned)n_strips * (unsigned)rows;     // row-units per system (< 2^31)

    // stage rings: the pad columns must read as zero for the whole launch
    {
        double2* q = smem + (size_t)Cfg::R * (Cfg::FCOLS + T);
        for (int e = i; e < Cfg::ring_rows * Cfg::SC; e += T) q[e] = make_double2(0.0, 0.0);
    }

    // ---- active systems and this CTA's range of row-units -------------------------------------------
    long long n_active = L.n_batch;
    int a_first = 0;
    long long start, end;
    if (BUDGETS) {
        const int q = (L.n_batch + T - 1) / T;            // systems scanned per thread
        const int s_lo = min(i * q, L.n_batch), s_hi = min(s_lo + q, L.n_batch);
        int cnt = 0;
        for (int s = s_lo; s < s_hi; ++s) cnt += sys_active(L, s, S) ? 1 : 0;
        int incl = cnt;                                   // inclusive scan over the CTA
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) {
            const int v = __shfl_up_sync(0xffffffffu, incl, o);
            if ((i & 31) >= o) incl += v;
        }
        if ((i & 31) == 31) sh.scan[i >> 5] = incl;
        __syncthreads();
        int base = 0, total = 0;
#pragma unroll
        for (int w = 0; w < T / 32; ++w) {
            if (w < (i >> 5)) base += sh.scan[w];
            total += sh.scan[w];
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
                if (sys_active(L, s, S)) {
                    if (a >= a_first && a <= a_last) sh.list[a - a_first] = s;
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
        const int sys = BUDGETS ? sh.list[a - a_first] : a;
        pos += Lr;
        sweep_segment<T, S, BUDGETS>(L, sys, strip, r0, Lr, n_strips, ups, smem, sh);
    }

    // ---- the last CTA of the launch advances the step counters of all systems that were active --------
    __threadfence();
    __syncthreads();
    if (i == 0) {
        const unsigned int prev = atomicAdd(L.gctl, 1u);
        sh.flag = (prev + 1u == gridDim.x) ? 1u : 0u;
    }
    __syncthreads();
    if (sh.flag) {
        __threadfence();
        for (int s = i; s < L.n_batch; s += T)
            if (sys_active(L, s, S)) {
                L.ss[s].k += S; L.ss[s].buf ^= 1;
                if (L.ss[s].phase == 3) L.ss[s].phase = 2;
            }
        if (i == 0) *L.gctl = 0u;
    }
}

}  // namespace bte
