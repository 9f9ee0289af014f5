// bte_regsweep.cuh -- the production streaming kernel of libbte_b200 (sm_100a): S leap-frog steps per pass
// over the lattice as a WARP-LEVEL SYSTOLIC PIPELINE of time steps.
//
// One launch = S consecutive leap-frog steps (eq. 40-41) of every active system = NS = 2 S applications of T
// (eq. 38), alternating whole / fractional grid, in one pass over the lattice: 64/S bytes of HBM traffic per
// lattice point per time step (ping-pong buffers), as in bte_sweep.cuh.  What differs is how the intermediate
// time levels travel.  bte_sweep.cuh keeps one thread per column, runs all NS stages in it and passes every
// stage row between threads through shared-memory rings behind one CTA-wide barrier per row (72 B of
// shared-memory traffic per half-update: that pipe and the barrier were its bound, profiles/r01e).  Here:
//
// * a strip of 32 K adjacent phi_y columns belongs to a team of S warps; lane l of every warp of the team holds
//   the K adjacent columns K l .. K l + K - 1;
// * warp ("role") s of the team performs leap-frog step s of the pass -- stages j = 2s (whole grid) and 2s + 1
//   (fractional grid) -- on a stream of rows: per iteration rho it takes one record
//       A = X^{j-1}[rho - j + 2]  (own pairs of stage j),   B = X^j[rho - j + 1]  (stencil row of stage j,
//                                                                own pairs of stage j + 1)
//   and emits one record (X^{j+1}[rho - j], X^{j+2}[rho - j - 1]) for role s + 1.  Role 0 gets its records from
//   HBM (cp.async into a ring, DPRE rows ahead, zero fill = boundary conditions (22)-(23)), role S-1 stores its
//   results to HBM;
// * inside a warp everything is registers: stage j + 1 takes the phi_y-difference of the row stage j has just
//   formed (its own K columns; the two outer neighbours by warp shuffle), so a stage lags its predecessor by ONE
//   row.  The update of a point is split in two (cn_partial / cn_complete, bte_device.cuh): when row n + 1 of the
//   stencil grid appears, its difference D finishes row n (started two iterations ago) and, with the own pair of
//   row n + 2 from the same record, starts row n + 2.  The only state a warp carries between iterations is the
//   partial right-hand side (Pg, Ph) of the two rows in flight per stage and column;
// * records travel between consecutive roles through a per-lane FIFO in shared memory: lane l of the producer
//   writes, lane l of the consumer reads (no cross-lane traffic, conflict-free 128-bit accesses), 64 B per point
//   per leap-frog step = 32 B of shared-memory traffic per half-update.  Flow control is two counters per lane
//   (records produced / consumed) in shared memory, polled only when the cached value runs out.  No CTA barrier,
//   no warp barrier, no fence: a lane's shared-memory accesses are performed in program order (the same
//   guarantee ptxas relies on when it lowers ld.acquire.cta.shared to a plain LDS and mbarrier.arrive.release.cta
//   to STS + SYNCS.ARRIVE without MEMBAR).
//
// The first / last HALO = NS - 1 columns of a strip are recomputed halos (W = 32 K - 2 HALO owned columns);
// segments that cut a column at an arbitrary row recompute HALO halo rows on each side (trapezoid in n as in m).
// Work decomposition: bands of STRIPS adjacent strips; band-rows (system, band, n) are numbered consecutively and
// dealt out in equal contiguous ranges to one CTA per SM; team g of the CTA takes strip g of the band, so the
// teams of a CTA touch adjacent 1 KB runs of every row (DRAM page locality).
// Per-step reductions (eq. 12, 17, 20): role s sees rows 0 and 1 of the new whole grid of step s -> per-strip
// partial sums -> fixed-order fold by the warp that completes a system (fold_sweep, bte_sweep.cuh).
#pragma once
#include <type_traits>

#include "bte_sweep.cuh"

namespace bte {

template <int S, int K>
struct RegCfg {
    static constexpr int NS = 2 * S;            // half-updates (stages) per pass
    static constexpr int HALO = NS - 1;         // halo columns on each side of a strip, halo rows of a segment
    static constexpr int COLS = 32 * K;         // columns a team computes
    static constexpr int W = COLS - 2 * HALO;   // owned columns per strip
    static constexpr int STRIPS = (S == 2) ? 6 : 4;   // teams per CTA = strips per band
    static constexpr int WARPS = S * STRIPS;
    static constexpr int T = 32 * WARPS;
    static constexpr int DIN = 8;               // slots of the HBM input ring of role 0
    static constexpr int DPRE = 6;              // rows prefetched ahead (slot of record t + DPRE was read 2 iterations ago)
    static constexpr int DF = 4;                // slots of a FIFO between consecutive roles
    static constexpr int REC = 2 * K * 32 + 2;  // double2 per record.  FIFO: A[K][32], B[K][32] (+2 unused); HBM input ring
                                                // of role 0: A = COLS columns, B = COLS + 2 columns, natural column order
    static constexpr int TEAM_D2 = (DIN + (S - 1) * DF) * REC;     // double2 per team
    static constexpr int TEAM_FLAGS = (S - 1) * 2 * 32;            // u32 per team: produced[32], consumed[32] per FIFO
    static constexpr int MAX_SPAN = 64;         // distinct systems one CTA range may touch
    // shared memory: rings of all teams | counters of all teams | mbarriers of the input rings (DIN per team) | per-warp
    // reduction slots
    static constexpr size_t off_flags = (size_t)STRIPS * TEAM_D2 * 16;
    static constexpr size_t off_bars = off_flags + (size_t)STRIPS * TEAM_FLAGS * 4;
    static constexpr size_t off_accs = off_bars + (size_t)STRIPS * DIN * 8;
    static constexpr size_t smem_bytes = off_accs + (size_t)WARPS * 2 * 32 * 8;
    static_assert(W >= 8, "strip too narrow");
    static_assert((DIN & (DIN - 1)) == 0 && (DF & (DF - 1)) == 0 && DPRE + 2 <= DIN, "ring sizes");
};

struct RegShared {
    int scan[16];
    int list[64];
    unsigned int flag;
};

__device__ __forceinline__ double2 shfl_up_d2(double2 v) {
    double2 r;
    r.x = __shfl_up_sync(0xffffffffu, v.x, 1);
    r.y = __shfl_up_sync(0xffffffffu, v.y, 1);
    return r;
}
__device__ __forceinline__ double2 shfl_down_d2(double2 v) {
    double2 r;
    r.x = __shfl_down_sync(0xffffffffu, v.x, 1);
    r.y = __shfl_down_sync(0xffffffffu, v.y, 1);
    return r;
}
// Flow-control counters and FIFO records: every access is volatile (ptxas keeps volatile accesses of a thread in
// program order -- a plain ld.shared of a record was observed to be sunk below the "slot free" store), the polls
// are acquire loads (a plain LDS in SASS; later accesses may not be hoisted above them).
__device__ __forceinline__ unsigned lds_u32_acquire(unsigned addr) {
    unsigned v;
    asm volatile("ld.acquire.cta.shared.u32 %0, [%1];\n" : "=r"(v) : "r"(addr) : "memory");
    return v;
}
__device__ __forceinline__ void sts_u32_volatile(unsigned addr, unsigned v) {
    asm volatile("st.volatile.shared.u32 [%0], %1;\n" ::"r"(addr), "r"(v) : "memory");
}
__device__ __forceinline__ double2 lds_d2_volatile(unsigned addr) {
    double2 v;
    asm volatile("ld.volatile.shared.v2.f64 {%0, %1}, [%2];\n" : "=d"(v.x), "=d"(v.y) : "r"(addr) : "memory");
    return v;
}
__device__ __forceinline__ void sts_d2_volatile(unsigned addr, double2 v) {
    asm volatile("st.volatile.shared.v2.f64 [%0], {%1, %2};\n" ::"r"(addr), "d"(v.x), "d"(v.y) : "memory");
}
// ---- 1-D bulk copies (TMA engine, SASS UBLKCP) with mbarrier completion: the HBM input ring of role 0 ----
__device__ __forceinline__ void mbar_init(unsigned bar, unsigned count) {
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;\n" ::"r"(bar), "r"(count) : "memory");
}
__device__ __forceinline__ void mbar_arrive_expect_tx(unsigned bar, unsigned bytes) {
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;\n" ::"r"(bar), "r"(bytes) : "memory");
}
__device__ __forceinline__ bool mbar_try_wait(unsigned bar, unsigned parity) {
    unsigned ok;
    asm volatile(
        "{\n .reg .pred p;\n mbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n selp.u32 %0, 1, 0, p;\n}\n"
        : "=r"(ok)
        : "r"(bar), "r"(parity)
        : "memory");
    return ok != 0;
}
// global -> shared, `bytes` a multiple of 16, both addresses 16-byte aligned; completion is signalled on `bar`
__device__ __forceinline__ void bulk_g2s(unsigned dst, const void* src, unsigned bytes, unsigned bar) {
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];\n" ::"r"(dst),
                 "l"(src), "r"(bytes), "r"(bar)
                 : "memory");
}

// What one warp keeps about its place in the team's pipeline for the whole launch.
struct RegChan {
    unsigned in_ring;      // shared address of the ring this role reads (role 0: HBM input ring, DIN slots)
    unsigned out_ring;     // shared address of the FIFO this role writes (roles < S-1), this lane
    unsigned in_bars;      // role 0: shared address of the DIN mbarriers of the input ring
    unsigned in_flags;     // shared address of this lane's produced / consumed counters of the input FIFO (+0 / +128)
    unsigned out_flags;    // ... of the output FIFO
    unsigned t_in;         // records taken so far in this launch
    unsigned t_out;        // records emitted so far
    unsigned prod_seen;    // cached copy of the producer's counter
    unsigned cons_seen;    // cached copy of the consumer's counter
};

// One segment of one warp: system sys, strip, rows r0 .. r0+Lr-1, role = leap-frog step of the pass.
//
// Iteration rho of a role with stages j0 = 2 role (whole grid) and j0 + 1 (fractional grid):
//   stage j0     takes record rho = (A, B) and forms   Z0 = X^{j0+1}[rho - j0]
//   stage j0 + 1 works one record behind: from (Bp, Zp) = (B, Z0) of iteration rho - 1 it forms
//                Z1 = X^{j0+2}[rho - j0 - 2], and record rho - 1 = (Zp, Z1) is emitted.
// The one-iteration skew makes the two stages of an iteration independent of each other (twice the
// instruction-level parallelism of a warp); a segment takes rho_end - rho_start + 2 iterations.
template <int S, int K, bool FIRST, bool LAST>
__device__ __forceinline__ void regsweep_segment(const Layout& L, const int sys, const int strip, const int r0,
                                                 const int Lr, const int n_strips, const unsigned ups,
                                                 const int role, RegChan& ch, double* __restrict__ accs) {
    using Cfg = RegCfg<S, K>;
    constexpr int NS = Cfg::NS, HALO = Cfg::HALO, W = Cfg::W, REC = Cfg::REC;
    constexpr int DIN = Cfg::DIN, DPRE = Cfg::DPRE, DF = Cfg::DF;
    constexpr unsigned RB = REC * 16;                   // bytes per record
    const int lane = threadIdx.x & 31;
    const double2 zero = make_double2(0.0, 0.0);

    const SysConst c = L.sc[sys];
    const long long k = L.ss[sys].k;
    const int cur = L.ss[sys].buf, nxt = cur ^ 1;
    const int N = L.N, pitch = L.pitch;
    // the fractional grid of the same buffer sits Y elements further (Y < 2^30, checked by the host)
    const int Y = L.n_batch * (N + 1 + 2 * GHOST) * pitch;
    const int c0 = strip * W;
    const int col0 = c0 - HALO + K * lane;              // this lane's first column
    const int j0 = 2 * role;                            // this role's stages: j0 (whole grid), j0 + 1 (fractional)
    const double* __restrict__ cn0 = cn_ptr(L, sys);

    bool valid[K], own[K];
    double gdt[K], kap[K], hb[4][K];                    // beta^t_m dt/2 at this step's four half-step times (eq. 28-29)
    {
        // field at the four half-step times of leap-frog step k + role (C14): lane v evaluates E(t_k + (j0 + v) dt/2)
        const double Ev = (lane < 4) ? field_E(c, ((double)k + 0.5 * (double)(j0 + lane)) * L.dt) : 0.0;
        double E[4];
#pragma unroll
        for (int v = 0; v < 4; ++v) E[v] = __shfl_sync(0xffffffffu, Ev, v);
#pragma unroll
        for (int q = 0; q < K; ++q) {
            const int col = col0 + q, x = K * lane + q;
            valid[q] = (col >= 0) && (col < L.M1);
            own[q] = valid[q] && (x >= HALO) && (x < HALO + W);
            const double ph = valid[q] ? L.phi[(size_t)sys * pitch + col] : 0.0;
            gdt[q] = valid[q] ? __dmul_rn(L.gm[(size_t)sys * pitch + col], L.dt) : 0.0;
            kap[q] = valid[q] ? c.kappa_dt : 0.0;       // invalid columns: w = 0, src = 0, kappa = 0 => stay 0
#pragma unroll
            for (int v = 0; v < 4; ++v) hb[v][q] = __dmul_rn(__fma_rn(c.B, ph, E[v]), L.hd);
        }
    }

    // row ranges (trapezoid in n): stage j forms rows max(0, lo_base + j) .. min(N, hi_base - j)
    const int lo_base = r0 - HALO, hi_base = r0 + Lr - 1 + HALO;
    const int lo0 = max(0, lo_base + j0), hi0 = min(N, hi_base - j0);          // stage j0
    const int lo1 = max(0, lo_base + j0 + 1), hi1 = min(N, hi_base - j0 - 1);  // stage j0 + 1
    const int rho_start = max(0, lo_base) - 2;          // first / last record of the segment (the same for every role)
    const int rho_end = min(N, r0 + Lr - 1) + NS - 1;
    // steady state of this role: both stages finish a row and start a row, no special rows 0 / 1, stores in range,
    // a record is taken and one is emitted
    const int rho_s0 = max(j0 + max(max(lo0, 2), LAST ? r0 : 0), j0 + 2 + max(lo1, 1));
    const int rho_s1 = min(min(hi0 - 2 + j0, hi1 + j0), rho_end);

    // ---- role 0: HBM -> input ring ---------------------------------------------------------------------
    // record rho = (A = H^0 row rho + 2, columns c0 - HALO .. + COLS - 1;  B = F^0 row rho + 1, one column more on
    // each side), natural column order.  Lane 0 issues two bulk copies per record (TMA engine) DPRE records ahead;
    // completion arrives on the slot's mbarrier.  Columns outside [0, pitch) are not copied: those parts of the ring
    // are zeroed once per segment (boundary condition (22)-(23) in m; the pad columns M+1 .. pitch-1 are zero in HBM).
    // Rows outside the lattice / the segment's trapezoid are not copied either: the record reads as zero.
    const double2* __restrict__ Hin = state_ptr(L, cur, 0, sys);   // row 0, column 0
    const int rf_max = min(N, hi_base + 1), rh_max = min(N, hi_base);      // last F^0 / H^0 row needed
    const int wa = c0 - HALO, wb = wa - 1;              // first column of the A / B part of a record
    const int ca0 = max(0, wa), ca1 = min(pitch, wa + Cfg::COLS);
    const int cb0 = max(0, wb), cb1 = min(pitch, wb + Cfg::COLS + 2);
    const unsigned nA = (unsigned)(ca1 - ca0) * 16u, nB = (unsigned)(cb1 - cb0) * 16u;
    const unsigned dA = (unsigned)(ca0 - wa) * 16u, dB = (unsigned)(Cfg::COLS + cb0 - wb) * 16u;   // offsets in a record
    unsigned tpre = ch.t_in;                            // record counter of the prefetch
    int rpre = rho_start;                               // its iteration
    if (FIRST && (nA != Cfg::COLS * 16 || nB != (Cfg::COLS + 2) * 16)) {   // first / last strip of a row
        for (int e = lane; e < DIN * REC; e += 32) sts_d2_volatile(ch.in_ring + (unsigned)e * 16u, zero);
        asm volatile("fence.proxy.async.shared::cta;\n" ::: "memory");   // generic writes before the bulk copies' writes
    }
    __syncwarp();
    auto prefetch = [&]() {
        if (FIRST) {
            __syncwarp();                               // every lane is done with the record that lived in this slot
            if (lane == 0 && rpre <= rho_end) {
                const unsigned slot = tpre & (DIN - 1);
                const unsigned dst = ch.in_ring + slot * RB, bar = ch.in_bars + slot * 8;
                const bool okh = (unsigned)(rpre + 2) <= (unsigned)rh_max, okf = (unsigned)(rpre + 1) <= (unsigned)rf_max;
                mbar_arrive_expect_tx(bar, (okh ? nA : 0u) + (okf ? nB : 0u));
                if (okh) bulk_g2s(dst + dA, Hin + ((rpre + 2) * pitch + ca0), nA, bar);
                if (okf) bulk_g2s(dst + dB, Hin + (Y + (rpre + 1) * pitch + cb0), nB, bar);
            }
            ++tpre; ++rpre;
        }
    };
    if (FIRST) {
#pragma unroll
        for (int v = 0; v < DPRE; ++v) prefetch();
    }
    const unsigned a_lane = ch.in_ring + (unsigned)lane * (K * 16);                      // this lane's A columns
    const unsigned x_lane = ch.in_ring + (Cfg::COLS + (lane == 31 ? Cfg::COLS + 1 : 0)) * 16;   // lanes 0 / 31: extra F^0 column

    // ---- role S-1: results -> HBM ----------------------------------------------------------------------
    double2* __restrict__ Hout = state_ptr(L, nxt, 0, sys) + col0;
    double2* __restrict__ Fout = Hout + Y;

    double2 P[2][2][K];                                 // partial right-hand sides in flight: [stage][slot][column]
    double2 Zp[K], Bp[K];                               // Z0 and B of the previous iteration (inputs of stage j0 + 1)
#pragma unroll
    for (int q = 0; q < K; ++q) {
        P[0][0][q] = P[0][1][q] = P[1][0][q] = P[1][1][q] = zero;
        Zp[q] = Bp[q] = zero;
    }

    int rho = rho_start;
    double nd0 = (double)(rho - j0);                    // row finished by stage j0, as double
    int o_out = (rho - j0) * pitch;                     // its element offset (stores of role S-1)
    const double* cnp = cn0 + (rho - j0 + 2);           // c_n of the row started by stage j0 (stage j0 + 1: two rows back)

    // One stage: src = row n + 1 of the stencil grid, ownp = own pairs of row n + 2; finishes row n, starts row n + 2.
    auto stage = [&](auto edge_tag, auto par_tag, auto jl_tag, const double2* src, const double2* ownp, const int n,
                     const double nd, double2* Z, const double2 Fx) {
        constexpr bool EDGE = decltype(edge_tag)::value;
        constexpr int PAR = decltype(par_tag)::value;
        constexpr int jl = decltype(jl_tag)::value;
        bool comp = true, strt = true;
        if (EDGE) {
            const int lo = jl ? lo1 : lo0, hi = jl ? hi1 : hi0;
            comp = n >= lo && n <= hi;
            strt = n + 2 >= lo && n + 2 <= hi;
        }
        if (!EDGE || comp || strt) {
            // phi_y-difference of row n + 1 of the stencil grid: interior columns from registers, the two outer ones
            // from the adjacent lanes
            double2 Lv = shfl_up_d2(src[K - 1]), Rv = shfl_down_d2(src[0]);
            if (FIRST && jl == 0) {
                if (lane == 0) Lv = Fx;
                if (lane == 31) Rv = Fx;
            }
            double2 D[K];
#pragma unroll
            for (int q = 0; q < K; ++q) {
                const double2 r = (q + 1 < K) ? src[q + 1 < K ? q + 1 : 0] : Rv;
                const double2 l = (q > 0) ? src[q > 0 ? q - 1 : 0] : Lv;
                D[q].x = __dsub_rn(r.x, l.x);
                D[q].y = __dsub_rn(r.y, l.y);
            }
            if (comp) {
#pragma unroll
                for (int q = 0; q < K; ++q) {
                    const double2 Pq = EDGE ? P[jl][0][q] : P[jl][PAR][q];
                    Z[q] = cn_complete(Pq, D[q], __dmul_rn(nd, hb[jl + 2][q]), kap[q], L.nu, L.nu2);
                    if (EDGE && n == 0) Z[q].y = 0.0;                 // b_0 == 0 (eq. 23, C3)
                }
                const bool mine = !EDGE || (n >= r0 && n < r0 + Lr);
                if (LAST && mine) {                                   // the two newest time levels go to HBM
                    double2* out = jl ? Fout + (o_out - 2 * pitch) : Hout + o_out;
#pragma unroll
                    for (int q = 0; q < K; ++q)
                        if (own[q]) out[q] = Z[q];
                }
                if (EDGE && jl == 0 && mine && n <= 1) {              // whole grid of step k + role + 1: reductions
                    double v = 0.0;
#pragma unroll
                    for (int q = 0; q < K; ++q)
                        if (own[q]) v += (n == 0) ? Z[q].x : Z[q].y;
                    accs[n * 32 + lane] = v;
                    if (LAST && n == 1) {
#pragma unroll
                        for (int q = 0; q < K; ++q) {
                            if (own[q] && col0 + q == 0) L.ss[sys].edge[0] = fabs(Z[q].y);
                            if (own[q] && col0 + q == L.M1 - 1) L.ss[sys].edge[1] = fabs(Z[q].y);
                        }
                    }
                }
            } else {
#pragma unroll
                for (int q = 0; q < K; ++q) Z[q] = zero;              // outside the lattice / this segment's halo
            }
            if (EDGE) {
#pragma unroll
                for (int q = 0; q < K; ++q) P[jl][0][q] = P[jl][1][q];
            }
            if (strt) {
                const double cj = __ldg(cnp - 2 * jl);                // c_{n+2}
                const double nd2 = nd + 2.0;
#pragma unroll
                for (int q = 0; q < K; ++q) {
                    double2 lo = D[q];
                    if (EDGE && n + 2 == 1) lo.x *= 2.0;              // chi(1) = 2, eq. (11)
                    const double2 Pn = cn_partial(ownp[q], lo, __dmul_rn(nd2, hb[jl][q]), __dmul_rn(cj, gdt[q]),
                                                  kap[q], L.xi);
                    if (EDGE) P[jl][1][q] = Pn; else P[jl][PAR][q] = Pn;
                }
            }
        } else {
#pragma unroll
            for (int q = 0; q < K; ++q) {
                Z[q] = zero;
                P[jl][0][q] = P[jl][1][q];
            }
        }
    };

    // edge_tag: std::true_type = fill / drain iteration (row predicates, special rows 0 and 1);
    // par_tag: steady state only: which of the two queue slots is finished (and refilled) in this iteration
    auto body = [&](auto edge_tag, auto par_tag) {
        constexpr bool EDGE = decltype(edge_tag)::value;
        // ---- take record rho ----
        double2 A[K], B[K], Fx = zero;
        if (!EDGE || rho <= rho_end) {
            if (FIRST) {
                prefetch();
                const unsigned slot = ch.t_in & (DIN - 1);
                while (!mbar_try_wait(ch.in_bars + slot * 8, (ch.t_in / DIN) & 1u)) {}   // record rho has landed
                const unsigned src = a_lane + slot * RB;
                bool okh = true, okf = true;
                if (EDGE) { okh = (unsigned)(rho + 2) <= (unsigned)rh_max; okf = (unsigned)(rho + 1) <= (unsigned)rf_max; }
#pragma unroll
                for (int q = 0; q < K; ++q) {
                    A[q] = okh ? lds_d2_volatile(src + q * 16) : zero;
                    B[q] = okf ? lds_d2_volatile(src + (Cfg::COLS + 1 + q) * 16) : zero;
                }
                Fx = okf ? lds_d2_volatile(x_lane + slot * RB) : zero;
                ++ch.t_in;
            } else {
                while ((int)(ch.prod_seen - ch.t_in) <= 0) ch.prod_seen = lds_u32_acquire(ch.in_flags);
                const unsigned src = ch.in_ring + (unsigned)lane * 16u + (ch.t_in & (DF - 1)) * RB;
#pragma unroll
                for (int q = 0; q < K; ++q) {
                    A[q] = lds_d2_volatile(src + q * 512);
                    B[q] = lds_d2_volatile(src + (K + q) * 512);
                }
                ++ch.t_in;
                sts_u32_volatile(ch.in_flags + 128, ch.t_in);               // slot free again
            }
        } else {
#pragma unroll
            for (int q = 0; q < K; ++q) A[q] = B[q] = zero;
        }
        double2 Z0[K], Z1[K];
        stage(edge_tag, par_tag, std::integral_constant<int, 0>{}, B, A, rho - j0, nd0, Z0, Fx);
        stage(edge_tag, par_tag, std::integral_constant<int, 1>{}, Zp, Bp, rho - j0 - 2, nd0 - 2.0, Z1, Fx);
        // ---- emit record rho - 1 = (X^{j0+1} row rho - 1 - j0, X^{j0+2} row rho - 2 - j0) ----
        if (!LAST && (!EDGE || rho > rho_start)) {
            while ((int)(ch.t_out - ch.cons_seen) >= DF) ch.cons_seen = lds_u32_acquire(ch.out_flags + 128);
            const unsigned dst = ch.out_ring + (ch.t_out & (DF - 1)) * RB;
#pragma unroll
            for (int q = 0; q < K; ++q) {
                sts_d2_volatile(dst + q * 512, Zp[q]);
                sts_d2_volatile(dst + (K + q) * 512, Z1[q]);
            }
            ++ch.t_out;
            sts_u32_volatile(ch.out_flags, ch.t_out);
        }
#pragma unroll
        for (int q = 0; q < K; ++q) { Zp[q] = Z0[q]; Bp[q] = B[q]; }
        ++rho; nd0 += 1.0;
        o_out += pitch; ++cnp;
    };

    using P0 = std::integral_constant<int, 0>;
    using P1 = std::integral_constant<int, 1>;
    while (rho <= rho_end + 1 && rho < rho_s0) body(std::true_type{}, P0{});
    while (rho + 1 <= rho_s1) {                         // two iterations per trip: the queue slots alternate
        body(std::false_type{}, P0{});
        body(std::false_type{}, P1{});
    }
    while (rho <= rho_end + 1) body(std::true_type{}, P0{});

    // per-strip partial sums of row 0 (a) and row 1 (b) of the new whole grid of this role's step -> eq. (12), (20)
    const bool has0 = (r0 == 0), has1 = (r0 <= 1) && (r0 + Lr > 1);
    if (has0 || has1) {
        double* part = L.partial + (((size_t)role * L.n_batch + sys) * pitch + strip) * 2;
        if (has0) {
            const double v = warp_sum(accs[lane]);
            if (lane == 0) part[0] = v;
        }
        if (has1) {
            const double v = warp_sum(accs[32 + lane]);
            if (lane == 0) part[1] = v;
        }
    }
    // the warp that completes the last row-unit of this system (all S roles count) folds its partial sums
    __threadfence();
    __syncwarp();
    unsigned int last = 0;
    if (lane == 0) {
        const unsigned int prev = atomicAdd(&L.ss[sys].done, (unsigned int)Lr);
        last = (prev + (unsigned int)Lr == ups) ? 1u : 0u;
    }
    last = __shfl_sync(0xffffffffu, last, 0);
    if (last) {
        __threadfence();
        fold_sweep(L, sys, n_strips, k, S);
    }
}

// BUDGETS: some system has a step budget (n_steps_total > 0) => the active set is compacted on the fly.
template <int S, int K, bool BUDGETS>
__global__ void __launch_bounds__(RegCfg<S, K>::T, 1) regsweep_kernel(const __grid_constant__ Layout L) {
    using Cfg = RegCfg<S, K>;
    constexpr int W = Cfg::W, STRIPS = Cfg::STRIPS, T = Cfg::T, WARPS = Cfg::WARPS;
    static_assert(Cfg::MAX_SPAN == 64 && WARPS <= 16, "RegShared sizes");
    extern __shared__ double2 rs_smem[];
    __shared__ RegShared sh;

    const int i = threadIdx.x, warp = i >> 5, lane = i & 31;
    const int team = warp / S, role = warp - team * S;
    const int rows = L.N + 1;
    const int n_strips = (L.M1 + W - 1) / W;
    const int n_bands = (n_strips + STRIPS - 1) / STRIPS;
    const unsigned ups = (unsigned)S * (unsigned)n_strips * (unsigned)rows;   // row-units per system, every role counts
    const long long upb = (long long)n_bands * rows;                          // band-rows per system

    const unsigned smem0 = (unsigned)__cvta_generic_to_shared(rs_smem);
    const unsigned team_base = smem0 + (unsigned)team * (Cfg::TEAM_D2 * 16);
    const unsigned flags0 = smem0 + (unsigned)Cfg::off_flags + (unsigned)team * (Cfg::TEAM_FLAGS * 4);
    double* accs = (double*)((char*)rs_smem + Cfg::off_accs) + warp * 64;
    RegChan ch;
    ch.in_ring = team_base + (role == 0 ? 0u : (unsigned)(Cfg::DIN + (role - 1) * Cfg::DF) * (Cfg::REC * 16));
    ch.out_ring = team_base + (unsigned)(Cfg::DIN + role * Cfg::DF) * (Cfg::REC * 16) + (unsigned)lane * 16u;
    ch.in_bars = smem0 + (unsigned)Cfg::off_bars + (unsigned)team * (Cfg::DIN * 8);
    ch.in_flags = flags0 + (unsigned)(role > 0 ? role - 1 : 0) * 256u + (unsigned)lane * 4u;
    ch.out_flags = flags0 + (unsigned)(role < S - 1 ? role : 0) * 256u + (unsigned)lane * 4u;
    ch.t_in = 0; ch.t_out = 0; ch.prod_seen = 0; ch.cons_seen = 0;
    for (int e = i; e < STRIPS * Cfg::TEAM_FLAGS; e += T) sts_u32_volatile(smem0 + (unsigned)Cfg::off_flags + (unsigned)e * 4u, 0u);
    if (i < STRIPS * Cfg::DIN) mbar_init(smem0 + (unsigned)Cfg::off_bars + (unsigned)i * 8u, 1u);
    asm volatile("fence.mbarrier_init.release.cluster;\n" ::: "memory");

    // ---- active systems and this CTA's range of band-rows --------------------------------------------
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
            if (lane >= o) incl += v;
        }
        if (lane == 31) sh.scan[warp] = incl;
        __syncthreads();
        int base = 0, total = 0;
#pragma unroll
        for (int w = 0; w < WARPS; ++w) {
            if (w < warp) base += sh.scan[w];
            total += sh.scan[w];
        }
        n_active = total;
        const long long units = n_active * upb;
        const long long U = (units + gridDim.x - 1) / gridDim.x;
        start = min((long long)blockIdx.x * U, units);
        end = min(start + U, units);
        if (start < end) {
            a_first = (int)(start / upb);
            const int a_last = (int)((end - 1) / upb);
            int a = base + incl - cnt;                    // index of this thread's first active system
            for (int s = s_lo; s < s_hi; ++s) {
                if (sys_active(L, s, S)) {
                    if (a >= a_first && a <= a_last) sh.list[a - a_first] = s;
                    ++a;
                }
            }
        }
    } else {
        const long long units = n_active * upb;
        const long long U = (units + gridDim.x - 1) / gridDim.x;
        start = min((long long)blockIdx.x * U, units);
        end = min(start + U, units);
    }
    __syncthreads();   // counters zeroed, mbarriers initialised, list visible

    // ---- every warp walks the CTA's range segment by segment: its team's strip of the band, its role's step ----
    long long pos = start;
    while (pos < end) {
        const int a = (int)(pos / upb);
        const int rem = (int)(pos - (long long)a * upb);
        const int band = rem / rows;
        const int r0 = rem - band * rows;
        const int Lr = (int)min((long long)(rows - r0), end - pos);
        const int sys = BUDGETS ? sh.list[a - a_first] : a;
        const int strip = band * STRIPS + team;
        pos += Lr;
        if (strip < n_strips) {
            if (role == 0) regsweep_segment<S, K, true, false>(L, sys, strip, r0, Lr, n_strips, ups, role, ch, accs);
            else if (role == S - 1) regsweep_segment<S, K, false, true>(L, sys, strip, r0, Lr, n_strips, ups, role, ch, accs);
            else regsweep_segment<S, K, false, false>(L, sys, strip, r0, Lr, n_strips, ups, role, ch, accs);
        }
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
            if (sys_active(L, s, S)) { L.ss[s].k += S; L.ss[s].buf ^= 1; }
        if (i == 0) *L.gctl = 0u;
    }
}

}  // namespace bte
