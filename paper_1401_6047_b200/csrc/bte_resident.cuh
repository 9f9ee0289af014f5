// bte_resident.cuh -- on-chip time loop for lattices that fit the shared memory of the GPU (sm_100a).
//
// One launch = ALL n_steps leap-frog steps (eq. 40-41) of every system of the batch (one CTA or one thread-block
// cluster per system; clusters are independent, the hardware schedules them as SMs become free).  The phi_y axis is cut into G slabs of
// Wc columns; CTA g keeps its slab of BOTH grids (whole and fractional, all harmonics n = 0..N) in shared
// memory for the whole launch, with one halo column on each side and one zero ghost row above and below
// (the zero perimeter of PAPER.md:L278, i.e. eq. 22-23).  HBM is touched twice: the state is loaded at the
// start and stored at the end (in place: no ping-pong buffer is needed because nothing streams).
//
// A half-update T (eq. 38) of grid X with the stencil of grid S reads, per point, its own pair of X and the
// four diagonal neighbours of S (eq. 30-31), all in shared memory, and writes X in place.  The two slab-edge
// columns of the new X are pushed to the neighbouring CTAs, then ONE barrier ends the half-update:
//   MODE 0  G = 1            __syncthreads
//   MODE 1  G <= 16 CTAs     one thread-block cluster: edge columns go straight into the neighbour's shared
//                            memory (st.shared::cluster), barrier.cluster arrive.release / wait.acquire
//   MODE 2  G <= #SMs CTAs   cooperative launch (co-residency): a slab carries HB halo columns on each side and talks
//                            to its neighbours only every HB half-updates.  Between two exchanges half-update i =
//                            0 .. HB-1 of the group also updates HB-1-i halo columns on each side (redundantly with
//                            the neighbour: trapezoid in time), then the HB edge columns of both grids go through a
//                            small global (L2) buffer; a CTA waits only for its two neighbours (release-store of
//                            its own group counter, acquire-spin on theirs) -- no grid-wide barrier, and the L2
//                            handshake (~2-3 us: membar, visibility, fetch) is paid once per HB half-updates
// Observables.  The sums of eq. (12), (20) and the running sums of eq. (17) are linear in the per-slab sums
// A_g(k) = sum_{m in slab} a_{0,m}, B_g(k) = sum b_{1,m}: every CTA accumulates its own B_g(k), B_g(k) cos(w t_k),
// B_g(k) sin(w t_k) (an extra "service" warp does that, and E(t), off the critical path) and the slabs are
// added once, in a fixed order, at the end of the launch: no cross-CTA reduction per step.
#pragma once
#include "bte_kernels.cuh"

#ifndef BTE_RES_UNROLL
#define BTE_RES_UNROLL 1
#endif

namespace bte {

constexpr int RES_UNROLL = BTE_RES_UNROLL;   // rows of the column march per loop trip

struct ResidentArgs {
    int G;                 // slabs = CTAs
    int Wc;                // columns per slab (the last slab may hold fewer valid columns)
    int T;                 // compute threads per CTA (blockDim.x = T + 32: one more warp does the bookkeeping)
    long long n_steps;     // steps of this launch (>= 1); a system's step budget may end it earlier
    int HB;                // halo columns on each side of a slab (1; MODE 2: 1 .. RES_MAX_HALO)
    double2* halo;         // MODE 2: [parity 2][grid 2][G][side 2][HB][N+1] edge columns of exchange group `parity`
    double* cta_out;       // [n_batch][G][8] per-slab results at the end of the launch
    unsigned int* flag;    // MODE 2: [G] exchange groups completed by each CTA (zeroed by the host before a launch)
};

__device__ __forceinline__ unsigned cluster_map(unsigned smem_addr, unsigned cta_rank) {
    unsigned r;
    asm volatile("mapa.shared::cluster.u32 %0, %1, %2;\n" : "=r"(r) : "r"(smem_addr), "r"(cta_rank));
    return r;
}
__device__ __forceinline__ void st_cluster_d2(unsigned addr, double2 v) {
    asm volatile("st.shared::cluster.v2.f64 [%0], {%1, %2};\n" ::"r"(addr), "d"(v.x), "d"(v.y) : "memory");
}
__device__ __forceinline__ void cluster_barrier() {
    asm volatile("barrier.cluster.arrive.release.aligned;\n" ::: "memory");
    asm volatile("barrier.cluster.wait.acquire.aligned;\n" ::: "memory");
}
__device__ __forceinline__ unsigned ld_acquire_u32(const unsigned* p) {
    unsigned v;
    asm volatile("ld.acquire.gpu.global.u32 %0, [%1];\n" : "=r"(v) : "l"(p) : "memory");
    return v;
}
__device__ __forceinline__ void st_release_u32(unsigned* p, unsigned v) {
    asm volatile("st.release.gpu.global.u32 [%0], %1;\n" ::"l"(p), "r"(v) : "memory");
}


constexpr int RES_MAX_HALO = 4;

// Shared memory of one CTA: Hs, Fs: [(N+3)][P] double2 with P = Wc + 2 HB (HB halo columns on each side, ghost rows
// 0 and N+2); then ph[P], gdt[P], cn[N+1] doubles.
__host__ __device__ inline size_t resident_smem_bytes(int N, int Wc, int HB = 1) {
    const size_t P = (size_t)Wc + 2 * (size_t)HB, rows = (size_t)N + 3;
    return 2 * rows * P * sizeof(double2) + (2 * P + (size_t)N + 1) * sizeof(double);
}

__device__ __forceinline__ double2 rlds_d2(unsigned addr) {
    double2 v;
    asm volatile("ld.shared.v2.f64 {%0, %1}, [%2];\n" : "=d"(v.x), "=d"(v.y) : "r"(addr));
    return v;
}
__device__ __forceinline__ void rsts_d2(unsigned addr, double2 v) {
    asm volatile("st.shared.v2.f64 [%0], {%1, %2};\n" ::"r"(addr), "d"(v.x), "d"(v.y) : "memory");
}
__device__ __forceinline__ double rlds_d(unsigned addr) {
    double v;
    asm volatile("ld.shared.f64 %0, [%1];\n" : "=d"(v) : "r"(addr));
    return v;
}

// One application of T (eq. 38) at point (n, j) of the slab: X updated in place with the stencil of S.
// Returns the new pair.  sX, sS: shared-memory addresses of the two arrays, both [(N+3)][P] with ghost rows and
// halo columns (no predicates); PB = P * 16 bytes; sph, sgdt, scn: addresses of the ph, gdt, c_n tables.
// j counts from the first halo column (own column jo sits at j = jo + HB).
__device__ __forceinline__ double2 resident_point(unsigned sX, unsigned sS, int n, int j, unsigned PB, unsigned sph,
                                                  unsigned sgdt, unsigned scn, const SysConst& c, const Layout& L,
                                                  double Ea, double Eb) {
    const unsigned off = (unsigned)(n + 1) * PB + (unsigned)j * 16;
    const unsigned up = sS + off - PB, dn = sS + off + PB;
    double2 lo, hi;
    {
        const double2 l = rlds_d2(up - 16), r = rlds_d2(up + 16);
        lo.x = __dsub_rn(r.x, l.x); lo.y = __dsub_rn(r.y, l.y);
        if (n == 1) lo.x *= 2.0;                   // chi(1) = 2, eq. (11)
    }
    {
        const double2 l = rlds_d2(dn - 16), r = rlds_d2(dn + 16);
        hi.x = __dsub_rn(r.x, l.x); hi.y = __dsub_rn(r.y, l.y);
    }
    const double ph = rlds_d(sph + (unsigned)j * 8);
    const double hba = __dmul_rn(__fma_rn(c.B, ph, Ea), L.hd);
    const double hbb = __dmul_rn(__fma_rn(c.B, ph, Eb), L.hd);
    const double src = __dmul_rn(rlds_d(scn + (unsigned)n * 8), rlds_d(sgdt + (unsigned)j * 8));
    double2 out = cn_point(rlds_d2(sX + off), lo, hi, (double)n, hba, hbb, src, c.kappa_dt, L.xi, L.nu, L.nu2);
    if (n == 0) out.y = 0.0;                       // b_0 == 0 (eq. 23, C3)
    rsts_d2(sX + off, out);
    return out;
}

// The same for rows nA .. nB-1 of ONE column (the grid mode's thread owns a column segment): marching over n, the
// phi_y-difference of a stencil row serves as the upper difference of row n and, two rows later, as the lower
// difference of row n + 2, and the per-column factors are formed once -- about half the instructions per point of
// resident_point (the grid mode is instruction-issue bound: profiles/r02b).  Same arithmetic, same rounding.
__device__ __forceinline__ void resident_column(unsigned sX, unsigned sS, int nA, int nB, int j, unsigned PB,
                                                unsigned sph, unsigned sgdt, unsigned scn, const SysConst& c,
                                                const Layout& L, double Ea, double Eb) {
    const double ph = rlds_d(sph + (unsigned)j * 8);
    const double hba = __dmul_rn(__fma_rn(c.B, ph, Ea), L.hd);
    const double hbb = __dmul_rn(__fma_rn(c.B, ph, Eb), L.hd);
    const double gdt = rlds_d(sgdt + (unsigned)j * 8);
    unsigned a = (unsigned)nA * PB + (unsigned)j * 16;          // row nA - 1 (array row index = n + 1)
    auto diff = [&](unsigned row_addr) {
        const double2 l = rlds_d2(sS + row_addr - 16), r = rlds_d2(sS + row_addr + 16);
        return make_double2(__dsub_rn(r.x, l.x), __dsub_rn(r.y, l.y));
    };
    double2 d0 = diff(a);                                       // row n - 1
    double2 d1 = diff(a + PB);                                  // row n
    unsigned cna = scn + (unsigned)nA * 8;
    double nd = (double)nA;
#pragma unroll RES_UNROLL
    for (int n = nA; n < nB; ++n) {
        a += PB;                                                // row n
        const double2 d2 = diff(a + PB);                        // row n + 1
        double2 lo = d0;
        if (n == 1) lo.x *= 2.0;                                // chi(1) = 2, eq. (11)
        const double src = __dmul_rn(rlds_d(cna), gdt);
        double2 out = cn_point(rlds_d2(sX + a), lo, d2, nd, hba, hbb, src, c.kappa_dt, L.xi, L.nu, L.nu2);
        if (n == 0) out.y = 0.0;                                // b_0 == 0 (eq. 23, C3)
        rsts_d2(sX + a, out);
        d0 = d1; d1 = d2;
        cna += 8; nd += 1.0;
    }
}

template <int MODE>
__global__ void __launch_bounds__(1024, 1) resident_kernel(const __grid_constant__ Layout L,
                                                           const __grid_constant__ ResidentArgs A) {
    extern __shared__ double2 smem[];
    // tables filled 32 entries at a time by the service warp, far ahead of their use (rings of 64):
    __shared__ double Es[64];             // E at half-step q of this launch (time (2 k0 + q) dt/2)       (C14)
    __shared__ double Cs[64], Sn[64];     // cos, sin of omega t at step s of this launch (t = (k0+s+1) dt) (C9)
    const int tid = threadIdx.x, T = A.T, NT = blockDim.x;
    const bool service = tid >= T;        // last warp: tables and the running sums, no lattice points
    const int lane = tid & 31, warp = tid >> 5;
    const int G = A.G, Wc = A.Wc;
    const int sys = blockIdx.x / G, g = blockIdx.x - sys * G;   // batches: one CTA / one cluster per system
    const int HB = (MODE == 2) ? A.HB : 1;   // halo columns on each side
    const int N = L.N, rows = N + 1, P = Wc + 2 * HB;
    const int c0 = g * Wc;
    const int Wv = min(Wc, L.M1 - c0);    // valid columns of this slab (>= HB by construction of the plan)

    double2* Hs = smem;
    double2* Fs = smem + (size_t)(N + 3) * P;
    double* phs = (double*)(Fs + (size_t)(N + 3) * P);
    double* gdts = phs + P;
    double* cns = gdts + P;

    const SysConst c = L.sc[sys];
    const long long k0 = L.ss[sys].k;
    const int buf = L.ss[sys].buf;
    // steps of this launch for this system: a step budget may end it early (uniform over the system's CTAs)
    const long long n_steps = c.n_steps_total > 0 ? max(0LL, min((long long)A.n_steps, c.n_steps_total - k0))
                                                  : (long long)A.n_steps;
    if (n_steps == 0) return;
    double2* __restrict__ Hg = state_ptr(L, buf, 0, sys);
    double2* __restrict__ Fg = state_ptr(L, buf, 1, sys);
    auto E_at = [&](long long q) {        // E at half-step q of this launch
        const long long v = 2 * k0 + q;
        return field_E(c, ((double)(v >> 1) + 0.5 * (double)(v & 1)) * L.dt);
    };
    auto csn_at = [&](long long s) {      // step s of this launch ends at t = (k0 + s + 1) dt
        double sn, cs;
        sincos(c.omega * ((double)(k0 + s + 1) * L.dt), &sn, &cs);
        Cs[s & 63] = cs; Sn[s & 63] = sn;
    };

    // ---- load: slab + halo columns straight from HBM; ghost rows / columns outside [0, M] are zero ----------
    const double2 zero = make_double2(0.0, 0.0);
    for (int e = tid; e < (N + 3) * P; e += NT) {
        const int r = e / P, jj = e - r * P;
        const int n = r - 1, col = c0 - HB + jj;
        const bool in = (n >= 0) && (n <= N) && (col >= 0) && (col < L.M1) && (jj < Wv + 2 * HB);
        Hs[e] = in ? Hg[(size_t)n * L.pitch + col] : zero;
        Fs[e] = in ? Fg[(size_t)n * L.pitch + col] : zero;
    }
    for (int j = tid; j < P; j += NT) {
        const int col = c0 - HB + j;
        const bool in = (col >= 0) && (col < L.M1) && (j < Wv + 2 * HB);
        phs[j] = in ? L.phi[(size_t)sys * L.pitch + col] : 0.0;
        gdts[j] = in ? __dmul_rn(L.gm[(size_t)sys * L.pitch + col], L.dt) : 0.0;
    }
    for (int n = tid; n < rows; n += NT) cns[n] = cn_ptr(L, sys)[n];
    for (int e = tid; e < 128; e += NT) {
        if (e < 64) Es[e] = E_at(e);
        else csn_at(e - 64);
    }
    __syncthreads();

    // this thread's points.  MODE 0 / 1: edge columns (jo = 0 and jo = Wv-1) first: e = T-1-tid, ... < nE (one point each,
    // pushed to the neighbours), then the interior columns 1 .. Wv-2.  MODE 2: all columns a group may ever update,
    // jo = -el .. Wv + er - 1 (el, er = HB - 1 where a neighbour exists); a half-update skips the columns beyond its reach.
    // Interior / MODE 2: thread = (column j_first of Wi, row chunk n_first): rows [nA, nB) of that column, marched over n.
    const int el = (MODE == 2 && g > 0) ? HB - 1 : 0, er = (MODE == 2 && g < G - 1) ? HB - 1 : 0;
    const int nE = (MODE == 2) ? 0 : (Wv >= 2 ? 2 : 1) * rows;
    const int Wi = (MODE == 2) ? Wv + el + er : max(Wv - 2, 0), nI = rows * Wi;
    const int wi = max(Wi, 1);
    int n_first = tid / wi, j_first = tid - n_first * wi;
    const int nch = max(T / wi, 1), Rr = (rows + nch - 1) / nch;
    int nA = min(n_first * Rr, rows), nB = min(nA + Rr, rows);
    // keep these in registers: without this the compiler re-derives them (integer divisions on the critical path of
    // every half-update) to save registers
    asm volatile("" : "+r"(n_first), "+r"(j_first), "+r"(nA), "+r"(nB));
    const unsigned sH = (unsigned)__cvta_generic_to_shared(Hs), sF = (unsigned)__cvta_generic_to_shared(Fs);
    const unsigned PB = (unsigned)P * 16;
    const unsigned sph = (unsigned)__cvta_generic_to_shared(phs), sgdt = (unsigned)__cvta_generic_to_shared(gdts),
                   scn = (unsigned)__cvta_generic_to_shared(cns);

    // service lane 0: this slab's share of the observables (fixed order in k => deterministic)
    double A_last = 0.0, B_last = 0.0, SV = 0.0, SC = 0.0, SS = 0.0;
    double window = L.ss[sys].window;     // advanced by repeated addition of dt, like the step-by-step kernels
    int sub = 0;                          // MODE 2: position of the half-update in its exchange group
    unsigned grp = 0;                     // MODE 2: exchange groups completed

    for (long long q = 0; q < 2 * n_steps; ++q) {
        const bool whole = (q & 1) == 0;
        if (service) {
            if (q > 0 && (q & 31) == 0) Es[(q + 32 + lane) & 63] = E_at(q + 32 + lane);
            if (!whole) {                          // the whole grid of step s was finished one phase ago
                const long long s = q >> 1;
                // sums of eq. (12), (20) over this slab, read from the whole grid (not written in this phase)
                double sa = 0.0, sb = 0.0;
                for (int j = lane; j < Wv; j += 32) {
                    sa += rlds_d2(sH + PB + (unsigned)(j + HB) * 16).x;          // a_{0,m}
                    sb += rlds_d2(sH + 2 * PB + (unsigned)(j + HB) * 16).y;      // b_{1,m}
                }
                sa = warp_sum(sa); sb = warp_sum(sb);
                if (lane == 0) {
                    A_last = sa; B_last = sb;
                    if (k0 + s + 1 > c.avg_start_step) {   // eq. (17), rectangle rule on whole-grid samples (C9)
                        SV += sb; SC += sb * Cs[s & 63]; SS += sb * Sn[s & 63]; window += L.dt;
                    }
                }
                __syncwarp();
                if (s > 0 && (s & 31) == 0) csn_at(s + 32 + lane);
            }
        } else {
            const unsigned sX = whole ? sH : sF, sS = whole ? sF : sH;
            const double Ea = Es[q & 63], Eb = Es[(q + 2) & 63];
            if (MODE != 2) {
                // slab-edge columns first: their new values go to the neighbours' halo columns.  Edge points are dealt
                // out from the LAST compute thread downwards, interior points from thread 0 upwards: with about one
                // point per thread no thread carries an edge point AND an interior point (the serial latency of a
                // half-update is one point update, not two).
                for (int e = T - 1 - tid; e < nE; e += T) {
                    const int side = e >= rows ? 1 : 0, n = e - side * rows;
                    const int j = side ? Wv - 1 : 0;
                    const double2 out = resident_point(sX, sS, n, j + 1, PB, sph, sgdt, scn, c, L, Ea, Eb);
                    if (MODE == 1) {
                        if (j == 0 && g > 0)
                            st_cluster_d2(cluster_map(sX + (unsigned)((n + 1) * P + Wc + 1) * 16, g - 1), out);
                        if (j == Wv - 1 && g < G - 1)
                            st_cluster_d2(cluster_map(sX + (unsigned)((n + 1) * P) * 16, g + 1), out);
                    }
                }
                // interior columns 1 .. Wv-2: this thread's column segment, marching over n
                if (nI > 0 && j_first < Wi && nA < nB)
                    resident_column(sX, sS, nA, nB, j_first + 2, PB, sph, sgdt, scn, c, L, Ea, Eb);
            } else {
                // half-update `sub` of the group: the slab and `reach` halo columns on each side (trapezoid in time)
                const int reach = HB - 1 - sub;
                const int jlo = el - min(reach, el), jhi = el + Wv + min(reach, er);   // in units of p's column index
                const bool xchg = (reach == 0) && (q + 1 < 2 * n_steps);   // this half-update ends an exchange group
                // pass 0: every column of this half-update; pass 2: all but the HB edge columns on each side
                // this thread's column j_first and rows [nA, nB) of it (fixed for the launch)
                auto sweep = [&](const int pass) {
                    const int j = j_first, jo = j - el;
                    const bool edge = (jo < HB) || (jo >= Wv - HB);
                    if ((j >= jlo) && (j < jhi) && (pass == 0 || !edge) && nA < nB)
                        resident_column(sX, sS, nA, nB, j + HB - el, PB, sph, sgdt, scn, c, L, Ea, Eb);
                };
                if (++sub == HB) sub = 0;
                if (!xchg) {
                    sweep(0);
                } else {
                    // ---- exchange: the HB edge columns of BOTH grids go to the neighbours.  The edge columns of this
                    // half-update are formed first and published while the interior is still being computed; the other
                    // grid (updated one half-update ago on the slab +- 1 column) is final already ----
                    ++grp;
                    // the 2 HB edge columns, dealt out one point per thread (about as many points as threads): the
                    // publication below then overlaps with the sweep over the rest of the slab
                    for (int e = tid; e < 2 * HB * rows; e += T) {
                        const int cc = e / rows, nn = e - cc * rows;               // cc < HB: left edge, else right edge
                        const int jo = cc < HB ? cc : Wv - 2 * HB + cc;
                        if (cc < HB || jo >= HB) resident_column(sX, sS, nn, nn + 1, jo + HB, PB, sph, sgdt, scn, c, L, Ea, Eb);
                    }
                    asm volatile("bar.sync 1, %0;\n" ::"r"(T) : "memory");   // compute warps: the edge columns are done
                    const int per = HB * rows;                 // elements per (grid, side)
                    double2* hb = A.halo + (size_t)(grp & 1u) * 2 * G * 2 * per;
                    // one warp per (grid, side, edge column), lanes over the rows: no index arithmetic per element
                    for (int task = warp; task < 4 * HB; task += (T >> 5)) {
                        const int gs = task / HB, cc = task - gs * HB;        // gs = grid * 2 + side
                        const int grid = gs >> 1, side = gs & 1;
                        const double2* Xs = (grid ? Fs : Hs) + P + HB + (side ? Wv - HB + cc : cc);
                        double2* dst = hb + ((size_t)(grid * G + g) * 2 + side) * per + cc * rows;
                        for (int nn = lane; nn < rows; nn += 32) dst[nn] = Xs[nn * P];
                    }
                    asm volatile("bar.sync 1, %0;\n" ::"r"(T) : "memory");
                    if (tid == 0) { __threadfence(); st_release_u32(A.flag + g, grp); }
                    sweep(2);
                    // wait for the two neighbours (one polling lane each), then fetch their edge columns into the halos
                    if (tid == 0 && g > 0) { while (ld_acquire_u32(A.flag + g - 1) < grp) {} }
                    if (tid == 32 && g < G - 1) { while (ld_acquire_u32(A.flag + g + 1) < grp) {} }
                    asm volatile("bar.sync 1, %0;\n" ::"r"(T) : "memory");
                    for (int task = warp; task < 4 * HB; task += (T >> 5)) {
                        const int gs = task / HB, cc = task - gs * HB;
                        const int grid = gs >> 1, side = gs & 1;      // side of MY slab the halo sits on
                        const int nb = side ? g + 1 : g - 1;
                        if (nb < 0 || nb >= G) continue;
                        // my left halo = the neighbour's RIGHT edge columns (its side 1), and vice versa
                        double2* Xs = (grid ? Fs : Hs) + P + (side ? HB + Wv + cc : cc);
                        const double2* src = hb + ((size_t)(grid * G + nb) * 2 + (side ? 0 : 1)) * per + cc * rows;
                        for (int nn = lane; nn < rows; nn += 32) Xs[nn * P] = __ldcg(src + nn);
                    }
                }
            }
        }
        // ---- end of the half-update -----------------------------------------------------------------------
        if (MODE == 1) cluster_barrier();
        else __syncthreads();
    }

    // ---- store: the slab goes back to the buffer it came from ------------------------------------------------
    for (int e = tid; e < rows * Wv; e += NT) {
        const int n = e / Wv, j = e - n * Wv;
        Hg[(size_t)n * L.pitch + c0 + j] = Hs[(n + 1) * P + j + HB];
        Fg[(size_t)n * L.pitch + c0 + j] = Fs[(n + 1) * P + j + HB];
    }
    if (g == 0 && tid == 0) L.ss[sys].edge[0] = fabs(Hs[2 * P + HB].y);               // |b_{1,0}|   (C12)
    if (g == G - 1 && tid == 0) L.ss[sys].edge[1] = fabs(Hs[2 * P + HB + Wv - 1].y);     // |b_{1,M}|
    if (service && lane == 0) {
        double* o = A.cta_out + (size_t)blockIdx.x * 8;
        o[0] = A_last; o[1] = B_last; o[2] = SV; o[3] = SC; o[4] = SS; o[5] = window;
    }
    // ---- one launch-wide synchronisation, then CTA 0 adds the slabs in a fixed order --------------------------
    const unsigned fin = 0x7fffffffu;     // larger than any group count
    if (MODE == 0) {
        __syncthreads();
    } else if (MODE == 1) {
        __threadfence();
        cluster_barrier();
    } else {
        __syncthreads();
        if (tid == 0) {
            __threadfence();
            st_release_u32(A.flag + g, fin);
        }
        if (g == 0 && warp == 0) {
            for (int s = lane; s < G; s += 32)
                while (ld_acquire_u32(A.flag + s) < fin) {
                }
            __threadfence();
        }
    }
    if (g == 0 && warp == 0) {
        double t[5] = {0.0, 0.0, 0.0, 0.0, 0.0};
        for (int s = lane; s < G; s += 32) {
#pragma unroll
            for (int x = 0; x < 5; ++x) t[x] += __ldcg(A.cta_out + ((size_t)sys * G + s) * 8 + x);
        }
#pragma unroll
        for (int x = 0; x < 5; ++x) t[x] = warp_sum(t[x]);
        if (lane == 0) {
            SysState* st = L.ss + sys;
            st->norm = c.norm_scale * t[0];                     // eq. (12)
            st->v_dr = c.v_scale * t[1];                        // eq. (20)
            st->sum_v += c.v_scale * t[2] * L.dt;               // eq. (17) sums, C9
            st->sum_c += c.v_scale * t[3] * L.dt;
            st->sum_s += c.v_scale * t[4] * L.dt;
            st->window = __ldcg(A.cta_out + (size_t)sys * G * 8 + 5);
            st->edge_leak = ((volatile double*)st->edge)[0] + ((volatile double*)st->edge)[1];
            st->k = k0 + n_steps;
        }
    }
}

}  // namespace bte
