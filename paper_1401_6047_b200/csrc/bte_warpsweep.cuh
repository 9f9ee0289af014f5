// bte_warpsweep.cuh -- streaming kernel of libbte_b200 (sm_100a): S leap-frog steps per pass over the lattice,
// every warp an independent register-resident pipeline of all 2 S half-updates.
//
// One launch = S consecutive leap-frog steps (eq. 40-41) of every active system = NS = 2 S applications of T
// (eq. 38), alternating whole / fractional grid, in one pass over the lattice: 64/S bytes of HBM traffic per
// lattice point per time step (ping-pong buffers), as in bte_sweep.cuh.  What differs is where the intermediate
// time levels live.  bte_sweep.cuh passes every stage row between the threads of a CTA through shared-memory rings
// behind one CTA-wide barrier per row (72 B of shared-memory traffic per half-update: that pipe and the barrier are
// its bound, profiles/r01e).  Here nothing but the HBM input ever touches shared memory:
//
// * a strip of 32 K adjacent phi_y columns belongs to ONE warp; lane l holds the K adjacent columns K l .. K l + K - 1
//   of every time level; the warp marches over n;
// * iteration rho: the warp takes one record from its input ring,
//       A = X^{-1}[rho + 2] (row of H^0: own pairs of stage 0),   B = X^0[rho + 1] (row of F^0: stencil row of stage 0)
//   and runs the NS stages one after the other, all in registers: stage j takes the phi_y-difference D of row
//   rho - j + 1 of X^j (its own K columns; the two outer neighbours by warp shuffle), which FINISHES row rho - j of
//   X^{j+1} (started two iterations ago) and, with the own pairs X^{j-1}[rho - j + 2] that stage j - 2 has formed in
//   this very iteration, STARTS row rho - j + 2 (cn_apply / cn_partial, bte_device.cuh).  The only state carried
//   between iterations is the partial right-hand side (Pg, Ph) of the two rows in flight per stage and column: it
//   lives in TENSOR MEMORY (tcgen05.alloc once per CTA; tcgen05.st.x2 per value, tcgen05.ld.x16 per stage: a per-warp
//   scratchpad of 2 NS slots, 6 x the shared-memory bandwidth on a path of its own), which frees 16 K registers per
//   stage pair and is what makes K = 3 columns per lane fit;
// * no barrier, no flag, no fence anywhere in the march: warps never exchange data.  The first / last HALO = NS - 1
//   columns of a strip are recomputed halos (W = 32 K - 2 HALO owned columns); segments that cut a column at an
//   arbitrary row recompute HALO halo rows on each side (trapezoid in n as in m) with the UNPREDICATED loop body (what
//   a stage forms outside its range is used by nobody; only the stores are limited to the segment's rows); predicated
//   iterations remain at rows 0, 1 and beyond N of the lattice;
// * HBM -> shared memory: one elected lane issues two 1-D bulk copies per record (TMA engine, SASS UBLKCP) DPRE records
//   ahead into a per-warp ring, completion on the slot's mbarrier; zero rows / columns outside the lattice are never read
//   (boundary conditions (22)-(23)).  The record of iteration rho + 1 is taken into registers at the END of iteration
//   rho (its ring reads hide behind the loop edge).  Results go to HBM straight from registers (128-bit stores).  With
//   EB = 8 the rows in HBM are fp32 pairs (bte_grid.precision 1): widened at the ring read, rounded once at the store;
// * mu^t_{n,m} = n beta^t_m dt/2 (eq. 28-29) is formed as fma(n, B phi_m dt/2, n E(t) dt/2): the column part is two
//   registers per column, the field part one number per row and half-step time (E(t_v) dt/2 sits in shared memory,
//   read as a broadcast), so that no per-column table of the NS + 2 half-step times is needed -- registers are for
//   the NS x 2 x K partial right-hand sides.  mu of row n at time t_v is the implicit mu' of stage v - 2 and the
//   explicit mu of stage v in the same iteration: formed once.
//
// Work decomposition: the (active system, strip) pairs are numbered consecutively and grouped into bands of WARPS; the
// band-rows (band, n) are dealt out in contiguous ranges of equal COST to one CTA per SM; warp g of the CTA takes pair g
// of the band, so the warps of a CTA touch adjacent 1.5 KB runs of every row (DRAM page locality), and a batch of narrow
// systems fills every warp.
// Per-step reductions (eq. 12, 17, 20): the even stages see rows 0 and 1 of the new whole grids -> per-strip partial
// sums -> fixed-order fold by the warp that completes a system (fold_sweep, bte_sweep.cuh).
#pragma once
#include <type_traits>

#include "bte_sweep.cuh"

// Tuning constants (compile-time; the defaults are the measured optimum on B200, DESIGN.md 5.1a / section 10):
//   (S = 2, 3, 4 steps per pass are instantiated; bte.cu picks 4 for long columns, else 3)
//   WARPS 8 (two per SMSP: 254 registers each), K 3 columns per lane, DIN 4 ring slots, CG 3 stages per coefficient
//   group, COVER 4 (a segment is charged COVER * NS / 2 = 2 NS row-iterations in the partition), TMSLOT 0 = automatic
#ifndef BTE_WS_WARPS
#define BTE_WS_WARPS 8
#endif
#ifndef BTE_WS_K
#define BTE_WS_K 3
#endif
#ifndef BTE_WS_DIN
#define BTE_WS_DIN 4
#endif
#ifndef BTE_WS_TMSLOT
#define BTE_WS_TMSLOT 0
#endif
#ifndef BTE_WS_COVER
#define BTE_WS_COVER 4
#endif
#ifndef BTE_WS_CG
#define BTE_WS_CG 3
#endif

namespace bte {

// EB: bytes of one stored (a, b) pair: 16 (fp64 state) or 8 (fp32 storage, bte_grid.precision 1; arithmetic stays fp64)
template <int S, int K, int EB = 16>
struct WarpCfg {
    static constexpr int NS = 2 * S;            // half-updates (stages) per pass
    static constexpr int NV = NS + 2;           // half-step times of a pass
    static constexpr int HALO = NS - 1;         // halo columns on each side of a strip, halo rows of a segment
    static constexpr int COLS = 32 * K;         // columns a warp computes
    static constexpr int W = COLS - 2 * HALO;   // owned columns per strip
    static constexpr int WARPS = BTE_WS_WARPS;             // warps per CTA = strips per band
    static constexpr int T = 32 * WARPS;
    static constexpr int DIN = BTE_WS_DIN;      // slots of the HBM input ring
    static constexpr int DPRE = DIN - 2;              // rows prefetched ahead (the slot of record t + DPRE was read 2 iterations ago)
    static constexpr int AX = EB == 8 ? 1 : 0;  // fp32 pairs: the A part starts one column early (16-byte alignment of the copies)
    static constexpr int ACOLS = COLS + 2 * AX; // columns of the A part of a record
    static constexpr int REC = ACOLS + COLS + 2; // pairs per record: A = ACOLS columns, B = COLS + 2 columns, natural order
    static constexpr int CG = BTE_WS_CG < 2 * S ? BTE_WS_CG : 2 * S;   // stages whose coefficients are formed together
    static constexpr int MAX_SPAN = 64;         // distinct systems one CTA range may touch
    // tensor memory: warp w owns the 32 lanes of quadrant w % 4, columns (w / 4) * TM_COLS .. + 2 NS TM_SLOT - 1;
    // one slot = the K pairs (4 K 32-bit columns, rounded to a power of two) of one stage and one iteration parity
    static constexpr int TM_SLOT = BTE_WS_TMSLOT ? BTE_WS_TMSLOT : (K <= 2 ? 8 : 16);
    static constexpr int TM_COLS = 2 * NS * TM_SLOT;
    static constexpr int TM_NEED = ((WARPS + 3) / 4) * TM_COLS;
    static constexpr int TM_ALLOC = TM_NEED <= 32 ? 32 : TM_NEED <= 64 ? 64 : TM_NEED <= 128 ? 128 : TM_NEED <= 256 ? 256 : 512;
    static_assert(4 * K <= TM_SLOT && TM_NEED <= 512, "tensor memory budget");
    // shared memory of one warp: input ring | E(t_v) dt/2 at the NV half-step times | mbarriers | reduction slots [S][2][32]
    static constexpr size_t off_tab = (size_t)DIN * REC * EB;
    static constexpr size_t off_bars = off_tab + (size_t)NV * 8;
    static constexpr size_t off_accs = off_bars + (size_t)DIN * 8;
    static constexpr size_t warp_bytes = off_accs + (size_t)S * 2 * 32 * 8;
    static constexpr size_t smem_bytes = (size_t)WARPS * warp_bytes;
    static_assert(W >= 8, "strip too narrow");
    static_assert((DIN & (DIN - 1)) == 0 && DPRE + 2 <= DIN, "ring sizes");
    static_assert(warp_bytes % 16 == 0 && off_tab % 16 == 0, "alignment");
};

struct WarpShared {
    int scan[16];
    int list[64];
    unsigned int flag;
    unsigned int tmem_base;
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
__device__ __forceinline__ double2 lds_d2_volatile(unsigned addr) {
    double2 v;
    asm volatile("ld.volatile.shared.v2.f64 {%0, %1}, [%2];\n" : "=d"(v.x), "=d"(v.y) : "r"(addr) : "memory");
    return v;
}
__device__ __forceinline__ void sts_d2_volatile(unsigned addr, double2 v) {
    asm volatile("st.volatile.shared.v2.f64 [%0], {%1, %2};\n" ::"r"(addr), "d"(v.x), "d"(v.y) : "memory");
}
// one stored pair from the ring -> fp64 (fp32 storage: widened, exact)
template <int EB>
__device__ __forceinline__ double2 lds_pair(unsigned addr) {
    if constexpr (EB == 16) {
        return lds_d2_volatile(addr);
    } else {
        float2 v;
        asm volatile("ld.volatile.shared.v2.f32 {%0, %1}, [%2];\n" : "=f"(v.x), "=f"(v.y) : "r"(addr) : "memory");
        return make_double2((double)v.x, (double)v.y);
    }
}
template <int EB> struct PairOf { using type = double2; };
template <> struct PairOf<8> { using type = float2; };
__device__ __forceinline__ void st_pair(double2* p, double2 v) { *p = v; }
__device__ __forceinline__ void st_pair(float2* p, double2 v) { *p = make_float2((float)v.x, (float)v.y); }   // rounded once
// ---- 1-D bulk copies (TMA engine, SASS UBLKCP) with mbarrier completion: the HBM input ring ----
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

// ---- tensor memory as the warp's private scratchpad (tcgen05.st / tcgen05.ld, 32 lanes x 32-bit columns) ----
// A warp reaches the 32 TMEM lanes of its quadrant (warp % 4); the partial right-hand sides of the rows in flight live
// there instead of in registers (96 registers per thread at S = 3).  Measured on B200 (one SM): 744 B/clk loads,
// 1000 B/clk stores, 39 cycles load-to-use -- 6 x the shared-memory bandwidth, on a path of its own.
// one double per store: its register pair is the natural operand (wider stores want 4 or 8 consecutive registers,
// which ptxas gathers with moves)
__device__ __forceinline__ void tm_st_d(unsigned taddr, double a) {
    asm volatile("{\n .reg .b32 lo, hi;\n mov.b64 {lo, hi}, %1;\n tcgen05.st.sync.aligned.32x32b.x2.b32 [%0], {lo, hi};\n}\n" ::"r"(taddr), "d"(a)
                 : "memory");
}
__device__ __forceinline__ void tm_st_d2(unsigned taddr, double2 a) {
    tm_st_d(taddr, a.x);
    tm_st_d(taddr + 2u, a.y);
}
template <int NR>
__device__ __forceinline__ void tm_ld(unsigned taddr, unsigned (&r)[NR]) {
    static_assert(NR == 8 || NR == 12 || NR == 16, "x8, x8 + x4 or x16");
    if constexpr (NR == 12) {
        asm volatile("tcgen05.ld.sync.aligned.32x32b.x8.b32 {%0,%1,%2,%3,%4,%5,%6,%7}, [%8];\n"
                     : "=r"(r[0]), "=r"(r[1]), "=r"(r[2]), "=r"(r[3]), "=r"(r[4]), "=r"(r[5]), "=r"(r[6]), "=r"(r[7])
                     : "r"(taddr)
                     : "memory");
        asm volatile("tcgen05.ld.sync.aligned.32x32b.x4.b32 {%0,%1,%2,%3}, [%4];\n"
                     : "=r"(r[8]), "=r"(r[9]), "=r"(r[10]), "=r"(r[11])
                     : "r"(taddr + 8u)
                     : "memory");
    } else if constexpr (NR == 8) {
        asm volatile("tcgen05.ld.sync.aligned.32x32b.x8.b32 {%0,%1,%2,%3,%4,%5,%6,%7}, [%8];\n"
                     : "=r"(r[0]), "=r"(r[1]), "=r"(r[2]), "=r"(r[3]), "=r"(r[4]), "=r"(r[5]), "=r"(r[6]), "=r"(r[7])
                     : "r"(taddr)
                     : "memory");
    } else {
        asm volatile("tcgen05.ld.sync.aligned.32x32b.x16.b32 {%0,%1,%2,%3,%4,%5,%6,%7,%8,%9,%10,%11,%12,%13,%14,%15}, [%16];\n"
                     : "=r"(r[0]), "=r"(r[1]), "=r"(r[2]), "=r"(r[3]), "=r"(r[4]), "=r"(r[5]), "=r"(r[6]), "=r"(r[7]),
                       "=r"(r[8]), "=r"(r[9]), "=r"(r[10]), "=r"(r[11]), "=r"(r[12]), "=r"(r[13]), "=r"(r[14]), "=r"(r[15])
                     : "r"(taddr)
                     : "memory");
    }
}
// the loaded registers may be read only after the wait: the wait takes them as in/out operands so that no use can be
// scheduled above it
template <int NR>
__device__ __forceinline__ void tm_wait_ld(unsigned (&r)[NR]) {
    if constexpr (NR == 8) {
        asm volatile("tcgen05.wait::ld.sync.aligned;\n"
                     : "+r"(r[0]), "+r"(r[1]), "+r"(r[2]), "+r"(r[3]), "+r"(r[4]), "+r"(r[5]), "+r"(r[6]), "+r"(r[7])::"memory");
    } else if constexpr (NR == 12) {
        asm volatile("tcgen05.wait::ld.sync.aligned;\n"
                     : "+r"(r[0]), "+r"(r[1]), "+r"(r[2]), "+r"(r[3]), "+r"(r[4]), "+r"(r[5]), "+r"(r[6]), "+r"(r[7]),
                       "+r"(r[8]), "+r"(r[9]), "+r"(r[10]), "+r"(r[11])::"memory");
    } else {
        asm volatile("tcgen05.wait::ld.sync.aligned;\n"
                     : "+r"(r[0]), "+r"(r[1]), "+r"(r[2]), "+r"(r[3]), "+r"(r[4]), "+r"(r[5]), "+r"(r[6]), "+r"(r[7]),
                       "+r"(r[8]), "+r"(r[9]), "+r"(r[10]), "+r"(r[11]), "+r"(r[12]), "+r"(r[13]), "+r"(r[14]), "+r"(r[15])::"memory");
    }
}
__device__ __forceinline__ void tm_wait_st() { asm volatile("tcgen05.wait::st.sync.aligned;\n" ::: "memory"); }

__device__ __forceinline__ bool elect_one() {
    unsigned ok;
    asm volatile("{\n .reg .pred p;\n elect.sync _|p, 0xffffffff;\n selp.u32 %0, 1, 0, p;\n}\n" : "=r"(ok));
    return ok != 0;
}
// a value every lane holds anyway, re-broadcast from lane 0: warp-uniform by construction whatever the compiler can
// prove about threadIdx (the operands of the bulk copies and of the tensor-memory accesses must be uniform; ptxas still
// keeps them in vector registers and converts with R2UR at the point of use)
__device__ __forceinline__ int uni(int v) { return __shfl_sync(0xffffffffu, v, 0); }
__device__ __forceinline__ unsigned uni(unsigned v) { return __shfl_sync(0xffffffffu, v, 0); }

// One segment of one warp: system sys, strip, rows r0 .. r0+Lr-1.
//   ring, bars: shared addresses of this warp's input ring and mbarriers; tabp: its table of E(t_v) dt/2; accs: its
//   reduction slots;
//   t_in: records taken so far in this launch (slot and mbarrier phase of the next one).
template <int S, int K, int EB>
__device__ __forceinline__ void warpsweep_segment(const Layout& L, const int sys, const int strip, const int r0,
                                                  const int Lr, const int n_strips, const unsigned ups,
                                                  const unsigned ring, double* tabp, const unsigned bars,
                                                  const unsigned tmP, double* __restrict__ accs, unsigned& t_in) {
    using Cfg = WarpCfg<S, K, EB>;
    using ST = typename PairOf<EB>::type;            // stored pair
    constexpr int NS = Cfg::NS, NV = Cfg::NV, HALO = Cfg::HALO, W = Cfg::W, REC = Cfg::REC, AX = Cfg::AX;
    constexpr int DIN = Cfg::DIN, DPRE = Cfg::DPRE;
    constexpr unsigned RB_BYTES = REC * EB;             // bytes per record
    const int lane = threadIdx.x & 31;
    const double2 zero = make_double2(0.0, 0.0);

    const SysConst c = L.sc[sys];
    const long long k = L.ss[sys].k;
    const int cur = uni(L.ss[sys].buf), nxt = cur ^ 1;
    const int N = L.N, pitch = L.pitch;
    // the fractional grid of the same buffer sits Y elements further (Y < 2^30, checked by the host)
    const int Y = L.n_batch * (N + 1 + 2 * GHOST) * pitch;
    const int c0 = strip * W;
    const int col0 = c0 - HALO + K * lane;              // this lane's first column
    const double* __restrict__ cn0 = cn_ptr(L, sys);

    bool own[K];
    double gdt[K], kap[K], bph[K];                      // a^(0) prefactor g_m dt, kappa, B phi_m dt/2 of this lane's columns
    {
        // field at the NV half-step times of the pass (C14): lane v evaluates E(t_k + v dt/2) dt/2
        if (lane < NV)
            *(volatile double*)(&tabp[lane]) = __dmul_rn(field_E(c, ((double)k + 0.5 * (double)lane) * L.dt), L.hd);
#pragma unroll
        for (int q = 0; q < K; ++q) {
            const int col = col0 + q, x = K * lane + q;
            const bool valid = (col >= 0) && (col < L.M1);
            own[q] = valid && (x >= HALO) && (x < HALO + W);
            bph[q] = valid ? __dmul_rn(__dmul_rn(c.B, L.phi[(size_t)sys * pitch + col]), L.hd) : 0.0;
            gdt[q] = valid ? __dmul_rn(L.gm[(size_t)sys * pitch + col], L.dt) : 0.0;
            kap[q] = valid ? c.kappa_dt : 0.0;          // invalid columns: w = 0, src = 0, kappa = 0 => stay 0
        }
        __syncwarp();
    }

    // row ranges (trapezoid in n): stage j forms rows max(0, lo_base + j) .. min(N, hi_base - j)
    const int lo_base = r0 - HALO, hi_base = r0 + Lr - 1 + HALO;
    const int rho_start = max(0, lo_base) - 2;          // first / last iteration of the segment
    const int rho_end = min(N, r0 + Lr - 1) + NS - 1;
    // Unpredicated ("steady") iterations: every stage finishes a row >= 2 and starts a row <= N of the LATTICE, records are
    // real rows.  The trapezoid of a segment that cuts a column in the middle needs no predicates: outside its range a
    // stage forms values nobody uses (from real rows and finite partial sums), only the stores are limited to the
    // segment's own rows.  Predicated iterations remain at the two ends of the lattice (rows 0, 1 and beyond N).
    const int rho_s0 = max(rho_start, NS + 1);
    const int rho_s1 = min(N - 2, rho_end);

    // ---- HBM -> input ring -------------------------------------------------------------------------------
    // record rho = (A = H^0 row rho + 2, columns c0 - HALO .. + COLS - 1;  B = F^0 row rho + 1, one column more on
    // each side), natural column order.  Columns outside [0, pitch) are not copied: those parts of the ring are
    // zeroed once per segment (boundary condition (22)-(23) in m; the pad columns M+1 .. pitch-1 are zero in HBM).
    // Rows outside the lattice / the segment's trapezoid are not copied either: the record reads as zero.
    const ST* __restrict__ Hin = (const ST*)L.state + (((size_t)cur * 2) * L.n_batch + sys) * grid_points(L) +
                                 (size_t)GHOST * pitch;   // whole grid of the live buffer: row 0, column 0
    const int rf_max = min(N, hi_base + 1), rh_max = min(N, hi_base);      // last F^0 / H^0 row needed
    const int wa = c0 - HALO - AX, wb = c0 - HALO - 1;  // first column of the A / B part of a record
    const int ca0 = max(0, wa), ca1 = min(pitch, wa + Cfg::ACOLS);
    const int cb0 = max(0, wb), cb1 = min(pitch, wb + Cfg::COLS + 2);
    const unsigned nA = (unsigned)(ca1 - ca0) * EB, nB = (unsigned)(cb1 - cb0) * EB;
    const unsigned dA = (unsigned)(ca0 - wa) * EB, dB = (unsigned)(Cfg::ACOLS + cb0 - wb) * EB;   // offsets in a record
    unsigned tpre = t_in;                               // record counter of the prefetch
    int rpre = rho_start;                               // its iteration
    if (nA != Cfg::ACOLS * EB || nB != (Cfg::COLS + 2) * EB) {   // first / last strip of a row
        for (int e = lane; e < DIN * REC * EB / 16; e += 32) sts_d2_volatile(ring + (unsigned)e * 16u, zero);
        asm volatile("fence.proxy.async.shared::cta;\n" ::: "memory");   // generic writes before the bulk copies' writes
    }
    __syncwarp();
    // Rows outside the lattice / the trapezoid are clamped to the nearest row the segment reads anyway (the record is
    // then read as zero, see `okh`, `okf` below): the prefetch is branch-free, two copies of fixed size per record.
    const ST* gA = Hin + ca0;
    const ST* gF = Hin + (Y + cb0);
    auto prefetch = [&]() {
        // (the record that lived in this slot was read two iterations ago: those loads have long been consumed)
        if (rpre <= rho_end && elect_one()) {
            const unsigned slot = tpre & (DIN - 1);
            const unsigned dst = ring + slot * RB_BYTES, bar = bars + slot * 8;
            mbar_arrive_expect_tx(bar, nA + nB);
            bulk_g2s(dst + dA, gA + min(max(rpre + 2, 0), rh_max) * pitch, nA, bar);
            bulk_g2s(dst + dB, gF + min(max(rpre + 1, 0), rf_max) * pitch, nB, bar);
        }
        ++tpre; ++rpre;
    };
#pragma unroll
    for (int v = 0; v < DPRE; ++v) prefetch();
    const unsigned a_lane = ring + (unsigned)(AX + K * lane) * EB;                        // this lane's A columns

    // ---- results -> HBM ----------------------------------------------------------------------------------
    ST* __restrict__ Hout = (ST*)L.state + (((size_t)nxt * 2) * L.n_batch + sys) * grid_points(L) + (size_t)GHOST * pitch + col0;
    ST* __restrict__ Fout = Hout + Y;

    // partial right-hand sides in flight: tensor memory, [stage][slot] x (K pairs = 8 columns of 32 bits); the slot
    // is the parity of the iteration (a row started in iteration rho is finished in iteration rho + 2)
    constexpr int SL = Cfg::TM_SLOT;
#pragma unroll
    for (int e = 0; e < 2 * NS * SL / 4; ++e) tm_st_d2(tmP + (unsigned)e * 4u, zero);

    int rho = rho_start;
    double nd0 = (double)rho;                           // row finished by stage 0, as double
    int o_out = (rho - (NS - 2)) * pitch;               // element offset of the row finished by stage NS - 2
    const double* cnp = cn0 + (rho + 2);                // c_n of the row started by stage 0 (stage j: j rows back)
    unsigned tmS = tmP;                                 // tensor-memory address of stage 0's slot of this iteration

    // take record r from the ring into registers (edge_tag: rows outside the lattice / the trapezoid read as zero)
    double2 RA[K], RB[K], RFL, RFR;
    // the answer of an mbarrier probe takes ~100 cycles: the probe for the next record is issued before the last
    // stage of an iteration (`probe`), its answer is looked at when the record is taken
    auto probe = [&]() { return mbar_try_wait(bars + (t_in & (DIN - 1)) * 8, (t_in / DIN) & 1u); };
    auto take = [&](auto edge_tag, const int r, bool landed) {
        constexpr bool EDGE = decltype(edge_tag)::value;
        const unsigned slot = t_in & (DIN - 1);
        while (!landed) landed = mbar_try_wait(bars + slot * 8, (t_in / DIN) & 1u);   // record r has landed
        const unsigned src = a_lane + slot * RB_BYTES;
        bool okh = true, okf = true;
        if (EDGE) { okh = (unsigned)(r + 2) <= (unsigned)rh_max; okf = (unsigned)(r + 1) <= (unsigned)rf_max; }
#pragma unroll
        for (int q = 0; q < K; ++q) {
            RA[q] = okh ? lds_pair<EB>(src + q * EB) : zero;
            RB[q] = okf ? lds_pair<EB>(src + (Cfg::ACOLS - AX + 1 + q) * EB) : zero;
        }
        RFL = okf ? lds_pair<EB>(src + (Cfg::ACOLS - AX) * EB) : zero;
        RFR = okf ? lds_pair<EB>(src + (Cfg::ACOLS - AX + 1 + K) * EB) : zero;
        ++t_in;
    };
    take(std::true_type{}, rho, false);

    // edge_tag: std::true_type = fill / drain iteration (row predicates, special rows 0 and 1)
    auto body = [&](auto edge_tag) {
        constexpr bool EDGE = decltype(edge_tag)::value;
        tm_wait_st();                                   // the partial sums stored in the previous iterations are in place
        // E(t_v) dt/2 of the NV half-step times: broadcast reads, issued here so that the prefetch code below covers
        // their latency (volatile: kept out of the loop-invariant registers)
        double Ev[NV];
#pragma unroll
        for (int v = 0; v < NV; ++v) Ev[v] = *(volatile double*)(&tabp[v]);
        unsigned Praw[SL];
        if (!EDGE) tm_ld(tmS, Praw);                    // stage 0's rows in flight
        // ---- record rho: taken at the end of the previous iteration (its ring reads are hidden behind the loop edge) ----
        double2 Z[NS + 2][K];                           // Z[j + 2] = output of stage j; Z[0] = A, Z[1] = B
#pragma unroll
        for (int q = 0; q < K; ++q) { Z[0][q] = RA[q]; Z[1][q] = RB[q]; }
        const double2 FL = RFL, FR = RFR;               // F^0 columns left / right of this lane's K columns
        prefetch();
        // mu[v][q] = n beta^{t_v}_m dt/2 of row n = rho - v + 2 (eq. 28-29): explicit mu of stage v, implicit mu' of stage v - 2
        double mu[NV][K];
        auto form_mu = [&](const int v) {
            const double ndv = nd0 + (double)(2 - v);
            const double ndE = __dmul_rn(ndv, Ev[v]);
#pragma unroll
            for (int q = 0; q < K; ++q) mu[v][q] = __fma_rn(ndv, bph[q], ndE);
        };
        // coefficients: they depend on (row, column, time) only, so the reciprocal chains are independent of each other
        // and of the data; they are formed for CG stages at a time (CG K independent chains side by side)
        bool landed = false;
        if (!EDGE) { form_mu(0); form_mu(1); }
        double2 pq[NS][K];                              // (nu, mu') / (nu^2 + mu'^2) of stage j
        auto form_coef = [&](const int j0) {
#pragma unroll
            for (int j = j0; j < j0 + Cfg::CG && j < NS; ++j) form_mu(j + 2);
#pragma unroll
            for (int j = j0; j < j0 + Cfg::CG && j < NS; ++j)
#pragma unroll
                for (int q = 0; q < K; ++q) pq[j][q] = cn_coef(mu[j + 2][q], L.nu, L.nu2);
        };
        if (!EDGE) form_coef(0);
#pragma unroll
        for (int j = 0; j < NS; ++j) {
            // src = Z[j + 1] = row n + 1 of the stencil grid X^j, ownp = Z[j] = own pairs of row n + 2;
            // finishes row n = rho - j of X^{j+1}, starts row n + 2
            const double2* src = Z[j + 1];
            const double2* ownp = Z[j];
            double2* Zo = Z[j + 2];
            const int n = rho - j;
            if (j == NS - 1) landed = probe();
            bool comp = true, strt = true;
            if (EDGE) {
                const int lo = max(0, lo_base + j), hi = min(N, hi_base - j);
                comp = n >= lo && n <= hi;
                strt = n + 2 >= lo && n + 2 <= hi;
            }
            if (EDGE) {
                // fill / drain and the ends of the lattice: a stage with neither a row to finish nor one to start costs
                // nothing (its output reads as zero); an active one fetches its own rows in flight and coefficients
                if (!(comp || strt)) {
#pragma unroll
                    for (int q = 0; q < K; ++q) Zo[q] = zero;
                    continue;
                }
                tm_ld(tmS + (unsigned)(j * 2 * SL), Praw);
                form_mu(j);
                form_mu(j + 2);
#pragma unroll
                for (int q = 0; q < K; ++q) pq[j][q] = cn_coef(mu[j + 2][q], L.nu, L.nu2);
            }
            // phi_y-difference of row n + 1 of the stencil grid: interior columns from registers, the two outer ones
            // from the adjacent lanes (stage 0: from the ring)
            double2 Lv, Rv;
            if (j == 0) { Lv = FL; Rv = FR; }
            else { Lv = shfl_up_d2(src[K - 1]); Rv = shfl_down_d2(src[0]); }
            if (!EDGE && (j + 1) % Cfg::CG == 0 && j + 1 < NS) form_coef(j + 1);   // while the shuffles are in flight
            // this stage's rows in flight have arrived; (steady state) ask for the next stage's
            tm_wait_ld(Praw);
            double2 Pq[K];
#pragma unroll
            for (int q = 0; q < K; ++q) {
                Pq[q].x = __hiloint2double((int)Praw[4 * q + 1], (int)Praw[4 * q]);
                Pq[q].y = __hiloint2double((int)Praw[4 * q + 3], (int)Praw[4 * q + 2]);
            }
            if (!EDGE && j + 1 < NS) tm_ld(tmS + (unsigned)((j + 1) * 2 * SL), Praw);
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
                    Zo[q] = cn_apply(Pq[q], D[q], kap[q], pq[j][q]);
                    if (EDGE && n == 0) Zo[q].y = 0.0;                // b_0 == 0 (eq. 23, C3)
                }
                const bool mine = (n >= r0 && n < r0 + Lr);
                if (j >= NS - 2 && mine) {                            // the two newest time levels go to HBM
                    ST* out = (j == NS - 1) ? Fout + (o_out - pitch) : Hout + o_out;
#pragma unroll
                    for (int q = 0; q < K; ++q)
                        if (own[q]) st_pair(out + q, Zo[q]);
                }
                if (EDGE && (j & 1) == 0 && mine && n <= 1) {         // whole grid of step k + j/2 + 1: reductions
                    double v = 0.0;
#pragma unroll
                    for (int q = 0; q < K; ++q)
                        if (own[q]) {                                 // (fp32 storage: the stored, rounded value)
                            const double z = (n == 0) ? Zo[q].x : Zo[q].y;
                            v += EB == 8 ? (double)(float)z : z;
                        }
                    accs[((j >> 1) * 2 + n) * 32 + lane] = v;
                    if (j == NS - 2 && n == 1) {
#pragma unroll
                        for (int q = 0; q < K; ++q) {
                            const double z = EB == 8 ? (double)(float)Zo[q].y : Zo[q].y;
                            if (own[q] && col0 + q == 0) L.ss[sys].edge[0] = fabs(z);
                            if (own[q] && col0 + q == L.M1 - 1) L.ss[sys].edge[1] = fabs(z);
                        }
                    }
                }
            } else {
#pragma unroll
                for (int q = 0; q < K; ++q) Zo[q] = zero;             // outside the lattice / this segment's halo
            }
            if (strt) {
                const double cj = __ldg(cnp - j);                     // c_{n+2}
#pragma unroll
                for (int q = 0; q < K; ++q) {
                    double2 lo = D[q];
                    if (EDGE && n + 2 == 1) lo.x *= 2.0;              // chi(1) = 2, eq. (11)
                    const double2 Pn = cn_partial(ownp[q], lo, mu[j][q], __dmul_rn(cj, gdt[q]), kap[q], L.xi);
                    tm_st_d2(tmS + (unsigned)(j * 2 * SL + q * 4), Pn);   // finished two iterations from now
                }
            }
        }
        ++rho; nd0 += 1.0;
        o_out += pitch; ++cnp;
        tmS = tmS == tmP ? tmP + (unsigned)SL : tmP;    // the other slot
        if (EDGE) { if (rho <= rho_end) take(edge_tag, rho, landed); }
        else take(edge_tag, rho, landed);               // steady state: the next record is a full one too
    };

    while (rho <= rho_end && rho < rho_s0) body(std::true_type{});
    while (rho < rho_s1) body(std::false_type{});      // (the record taken at its end must be a steady one too)
    while (rho <= rho_end) body(std::true_type{});

    // per-strip partial sums of row 0 (a) and row 1 (b) of the S new whole grids -> eq. (12), (20)
    const bool has0 = (r0 == 0), has1 = (r0 <= 1) && (r0 + Lr > 1);
    if (has0 || has1) {
        __syncwarp();
#pragma unroll
        for (int s = 0; s < S; ++s) {
            double* part = L.partial + (((size_t)s * L.n_batch + sys) * pitch + strip) * 2;
            if (has0) {
                const double v = warp_sum(accs[(s * 2 + 0) * 32 + lane]);
                if (lane == 0) part[0] = v;
            }
            if (has1) {
                const double v = warp_sum(accs[(s * 2 + 1) * 32 + lane]);
                if (lane == 0) part[1] = v;
            }
        }
    }
    // the warp that completes the last row-unit of this system folds its partial sums
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
template <int S, int K, bool BUDGETS, int EB>
__global__ void __launch_bounds__(WarpCfg<S, K, EB>::T, 1) warpsweep_kernel(const __grid_constant__ Layout L) {
    using Cfg = WarpCfg<S, K, EB>;
    constexpr int W = Cfg::W, WARPS = Cfg::WARPS, T = Cfg::T;
    static_assert(Cfg::MAX_SPAN == 64 && WARPS <= 16, "WarpShared sizes");
    extern __shared__ double2 ws_smem[];
    __shared__ WarpShared sh;

    const int i = threadIdx.x, lane = i & 31;
    const int warp = uni(i >> 5);
    const int rows = L.N + 1;
    const int n_strips = (L.M1 + W - 1) / W;
    const unsigned ups = (unsigned)n_strips * (unsigned)rows;                 // row-units per system
    // bands of WARPS consecutive (active system, strip) pairs: a band may straddle two systems of a batch
    auto bands_of = [&](const long long n_act) -> long long { return (n_act * n_strips + WARPS - 1) / WARPS; };

    const unsigned base = (unsigned)__cvta_generic_to_shared(ws_smem) + (unsigned)warp * (unsigned)Cfg::warp_bytes;
    const unsigned ring = base, bars = base + (unsigned)Cfg::off_bars;
    double* tabp = (double*)((char*)ws_smem + (size_t)warp * Cfg::warp_bytes + Cfg::off_tab);
    double* accs = (double*)((char*)ws_smem + (size_t)warp * Cfg::warp_bytes + Cfg::off_accs);
    unsigned t_in = 0;
    if (lane < Cfg::DIN) mbar_init(bars + (unsigned)lane * 8u, 1u);
    asm volatile("fence.mbarrier_init.release.cluster;\n" ::: "memory");
    if (warp == 0) {                                      // one CTA per SM (launch bounds, shared memory): no contention
        asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], %1;\n" ::"r"(
                         (unsigned)__cvta_generic_to_shared(&sh.tmem_base)), "r"(Cfg::TM_ALLOC) : "memory");
        asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;\n" ::: "memory");
    }
    asm volatile("tcgen05.fence::before_thread_sync;\n" ::: "memory");

    // ---- active systems and this CTA's range of band-rows --------------------------------------------
    // Static partition balanced by COST, not by rows: a segment costs its rows plus about 2 NS row-iterations of
    // pipeline fill / drain and halo rows (slower, predicated iterations), so a range that spans a band boundary must
    // get fewer rows.  Every band is charged c_over + rows cost units; the i-th boundary sits at cost i / gridDim.x
    // of the total (boundaries that fall into a band's overhead snap to the band's first row).
    auto range_cut = [&](const long long i, const long long nb) -> long long {
        // (c_over = 2 NS, measured: config 4 at S = 4 with 8 / 12 / 16 / 20 / 24 / 32 row-iterations: 181.5 / 184.0 / 184.3 /
        // 182.6 / 181.5 / 179.2 G; config 3 at S = 3 with 6 / 9 / 12 / 15 / 18 / 21: 132.9 / 133.7 / 136.3 / 135.8 / 135.5 / 134.9 G)
        const long long c_over = BTE_WS_COVER * Cfg::NS / 2, band_cost = rows + c_over;
        const long long y = (i * nb * band_cost) / gridDim.x;
        const long long b = y / band_cost, r = y - b * band_cost;
        return b * rows + min(max(r - c_over, 0LL), (long long)rows);
    };
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
        int base_a = 0, total = 0;
#pragma unroll
        for (int w = 0; w < WARPS; ++w) {
            if (w < warp) base_a += sh.scan[w];
            total += sh.scan[w];
        }
        n_active = total;
        start = range_cut(blockIdx.x, bands_of(n_active));
        end = range_cut(blockIdx.x + 1, bands_of(n_active));
        if (start < end) {
            a_first = (int)((start / rows) * WARPS / n_strips);
            const int a_last = (int)min(n_active - 1, (((end - 1) / rows) * WARPS + WARPS - 1) / n_strips);
            int a = base_a + incl - cnt;                  // index of this thread's first active system
            for (int s = s_lo; s < s_hi; ++s) {
                if (sys_active(L, s, S)) {
                    if (a >= a_first && a <= a_last) sh.list[a - a_first] = s;
                    ++a;
                }
            }
        }
    } else {
        start = range_cut(blockIdx.x, bands_of(n_active));
        end = range_cut(blockIdx.x + 1, bands_of(n_active));
    }
    __syncthreads();   // mbarriers initialised, list visible, tensor memory allocated
    asm volatile("tcgen05.fence::after_thread_sync;\n" ::: "memory");
    const unsigned tmP = uni(sh.tmem_base) + (((unsigned)(warp & 3) * 32u) << 16) + (unsigned)(warp >> 2) * Cfg::TM_COLS;

    // ---- every warp walks the CTA's range segment by segment: its strip of the band ----------------------
    long long pos = start;
    while (pos < end) {
        const long long band = pos / rows;
        const int r0 = (int)(pos - band * rows);
        const int Lr = (int)min((long long)(rows - r0), end - pos);
        const long long g = band * WARPS + warp;          // this warp's (active system, strip) pair
        pos += Lr;
        if (g < n_active * n_strips) {
            const int a = (int)(g / n_strips);
            const int strip = (int)(g - (long long)a * n_strips);
            const int sys = BUDGETS ? uni(sh.list[a - a_first]) : a;
            warpsweep_segment<S, K, EB>(L, sys, strip, r0, Lr, n_strips, ups, ring, tabp, bars, tmP, accs, t_in);
        }
    }

    // ---- the last CTA of the launch advances the step counters of all systems that were active --------
    tm_wait_st();
    asm volatile("tcgen05.fence::before_thread_sync;\n" ::: "memory");
    __threadfence();
    __syncthreads();
    if (warp == 0)
        asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, %1;\n" ::"r"(sh.tmem_base), "r"(Cfg::TM_ALLOC) : "memory");
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
