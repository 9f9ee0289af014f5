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
//   MODE 2  G <= #SMs CTAs   cooperative launch (co-residency): edge columns go through a small global (L2)
//                            buffer; a CTA waits only for its two neighbours (release-store of its own
//                            half-update counter, acquire-spin on theirs) -- no grid-wide barrier per step
// Observables.  The sums of eq. (12), (20) and the running sums of eq. (17) are linear in the per-slab sums
// A_g(k) = sum_{m in slab} a_{0,m}, B_g(k) = sum b_{1,m}: every CTA accumulates its own B_g(k), B_g(k) cos(w t_k),
// B_g(k) sin(w t_k) (an extra "service" warp does that, and E(t), off the critical path) and the slabs are
// added once, in a fixed order, at the end of the launch: no cross-CTA reduction per step.
#pragma once
#include "bte_kernels.cuh"

namespace bte {

struct ResidentArgs {
    int G;                 // slabs = CTAs
    int Wc;                // columns per slab (the last slab may hold fewer valid columns)
    int T;                 // compute threads per CTA (blockDim.x = T + 32: one more warp does the bookkeeping)
    long long n_steps;     // steps of this launch (>= 1); a system's step budget may end it earlier
    double2* halo;         // MODE 2: [grid 2][G][side 2][N+1] edge columns
    double* cta_out;       // [n_batch][G][8] per-slab results at the end of the launch
    unsigned int* flag;    // MODE 2: [G] half-updates completed by each CTA (zeroed by the host before a launch)
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


// Shared memory of one CTA: Hs, Fs: [(N+3)][P] double2 with P = Wc + 2 (halo columns 0 and Wv+1, ghost rows
// 0 and N+2); then ph[Wc], gdt[Wc], cn[N+1] doubles.
__host__ __device__ inline size_t resident_smem_bytes(int N, int Wc) {
    const size_t P = (size_t)Wc + 2, rows = (size_t)N + 3;
    return 2 * rows * P * sizeof(double2) + (2 * (size_t)Wc + (size_t)N + 1) * sizeof(double);
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
__device__ __forceinline__ double2 resident_point(unsigned sX, unsigned sS, int n, int j, unsigned PB, unsigned sph,
                                                  unsigned sgdt, unsigned scn, const SysConst& c, const Layout& L,
                                                  double Ea, double Eb) {
    const unsigned off = (unsigned)(n + 1) * PB + (unsigned)(j + 1) * 16;
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
    const int N = L.N, rows = N + 1, P = Wc + 2;
    const int c0 = g * Wc;
    const int Wv = min(Wc, L.M1 - c0);    // valid columns of this slab (>= 1 by construction of the plan)

    double2* Hs = smem;
    double2* Fs = smem + (size_t)(N + 3) * P;
    double* phs = (double*)(Fs + (size_t)(N + 3) * P);
    double* gdts = phs + Wc;
    double* cns = gdts + Wc;

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
        const int n = r - 1, col = c0 - 1 + jj;
        const bool in = (n >= 0) && (n <= N) && (col >= 0) && (col < L.M1) && (jj <= Wv + 1);
        Hs[e] = in ? Hg[(size_t)n * L.pitch + col] : zero;
        Fs[e] = in ? Fg[(size_t)n * L.pitch + col] : zero;
    }
    for (int j = tid; j < Wc; j += NT) {
        const bool in = j < Wv;
        phs[j] = in ? L.phi[(size_t)sys * L.pitch + c0 + j] : 0.0;
        gdts[j] = in ? __dmul_rn(L.gm[(size_t)sys * L.pitch + c0 + j], L.dt) : 0.0;
    }
    for (int n = tid; n < rows; n += NT) cns[n] = cn_ptr(L, sys)[n];
    for (int e = tid; e < 128; e += NT) {
        if (e < 64) Es[e] = E_at(e);
        else csn_at(e - 64);
    }
    __syncthreads();

    // this thread's points.  Edge columns (j = 0 and j = Wv-1) first: e = tid, tid + T, ... < nE;
    // then the interior columns 1 .. Wv-2: p = tid, tid + T, ... < rows * Wi, p = n * Wi + (j - 1)
    const int nE = (Wv >= 2 ? 2 : 1) * rows;
    const int Wi = max(Wv - 2, 0), nI = rows * Wi;
    const int wi = max(Wi, 1);
    int n_first = tid / wi, j_first = tid - n_first * wi;
    int dn = T / wi, dj = T - dn * wi;
    // keep the quotients in registers: without this the compiler re-derives them (an integer division on the
    // critical path of every half-update) to save four registers
    asm volatile("" : "+r"(n_first), "+r"(j_first), "+r"(dn), "+r"(dj));
    const unsigned sH = (unsigned)__cvta_generic_to_shared(Hs), sF = (unsigned)__cvta_generic_to_shared(Fs);
    const unsigned PB = (unsigned)P * 16;
    const unsigned sph = (unsigned)__cvta_generic_to_shared(phs), sgdt = (unsigned)__cvta_generic_to_shared(gdts),
                   scn = (unsigned)__cvta_generic_to_shared(cns);

    // service lane 0: this slab's share of the observables (fixed order in k => deterministic)
    double A_last = 0.0, B_last = 0.0, SV = 0.0, SC = 0.0, SS = 0.0;
    double window = L.ss[sys].window;     // advanced by repeated addition of dt, like the step-by-step kernels

    for (long long q = 0; q < 2 * n_steps; ++q) {
        const bool whole = (q & 1) == 0;
        double2* X = whole ? Hs : Fs;
        const unsigned done = (unsigned)q + 1u;
        if (service) {
            if (q > 0 && (q & 31) == 0) Es[(q + 32 + lane) & 63] = E_at(q + 32 + lane);
            if (!whole) {                          // the whole grid of step s was finished one phase ago
                const long long s = q >> 1;
                // sums of eq. (12), (20) over this slab, read from the whole grid (not written in this phase)
                double sa = 0.0, sb = 0.0;
                for (int j = lane; j < Wv; j += 32) {
                    sa += rlds_d2(sH + PB + (unsigned)(j + 1) * 16).x;          // a_{0,m}
                    sb += rlds_d2(sH + 2 * PB + (unsigned)(j + 1) * 16).y;      // b_{1,m}
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
            // slab-edge columns first: their new values go to the neighbours' halo columns.  Edge points are dealt
            // out from the LAST compute thread downwards, interior points from thread 0 upwards: with about one
            // point per thread no thread carries an edge point AND an interior point (the serial latency of a
            // half-update is one point update, not two).
            for (int e = T - 1 - tid; e < nE; e += T) {
                const int side = e >= rows ? 1 : 0, n = e - side * rows;
                const int j = side ? Wv - 1 : 0;
                const double2 out = resident_point(sX, sS, n, j, PB, sph, sgdt, scn, c, L, Ea, Eb);
                if (MODE == 1) {
                    if (j == 0 && g > 0)
                        st_cluster_d2(cluster_map(sX + (unsigned)((n + 1) * P + Wc + 1) * 16, g - 1), out);
                    if (j == Wv - 1 && g < G - 1)
                        st_cluster_d2(cluster_map(sX + (unsigned)((n + 1) * P) * 16, g + 1), out);
                } else if (MODE == 2) {
                    double2* hl = A.halo + ((size_t)((whole ? 0 : 1) * G + g) * 2) * rows;
                    if (j == 0) hl[n] = out;
                    if (j == Wv - 1) hl[rows + n] = out;
                }
            }
            if (MODE == 2) {
                // publish "edge columns of half-update q are out" while the interior is still being computed.
                // Named barrier over the compute warps only (the service warp does not take part).
                asm volatile("bar.sync 1, %0;\n" ::"r"(T) : "memory");
                if (tid == 0) { __threadfence(); st_release_u32(A.flag + g, done); }
            }
            int n = n_first, j = j_first;
            for (int p = tid; p < nI; p += T) {
                resident_point(sX, sS, n, j + 1, PB, sph, sgdt, scn, c, L, Ea, Eb);
                j += dj; n += dn;
                if (j >= wi) { j -= wi; ++n; }
            }
            if (MODE == 2) {
                // halo columns of X for the next half-update, fetched in chunks of 32 rows: chunk ch < nch is rows
                // 32 ch .. of the left halo, chunk nch + ch the same rows of the right halo.  One chunk per warp;
                // one lane polls the neighbour's counter ("edge columns of half-update q are out"), then every
                // lane fetches its element (one L2 round trip).
                const int nch = (rows + 31) >> 5;
                for (int ch = warp; ch < 2 * nch; ch += (T >> 5)) {
                    const int side = ch >= nch ? 1 : 0;
                    const int nb = side ? g + 1 : g - 1;
                    if (nb < 0 || nb >= G) continue;
                    if (lane == 0) {
                        while (ld_acquire_u32(A.flag + nb) < done) {
                        }
                    }
                    __syncwarp();
                    const int nn = ((ch - side * nch) << 5) + lane;
                    if (nn < rows)
                        X[(nn + 1) * P + (side ? Wv + 1 : 0)] =
                            __ldcg(A.halo + ((size_t)((whole ? 0 : 1) * G + nb) * 2 + (side ? 0 : 1)) * rows + nn);
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
        Hg[(size_t)n * L.pitch + c0 + j] = Hs[(n + 1) * P + j + 1];
        Fg[(size_t)n * L.pitch + c0 + j] = Fs[(n + 1) * P + j + 1];
    }
    if (g == 0 && tid == 0) L.ss[sys].edge[0] = fabs(Hs[2 * P + 1].y);          // |b_{1,0}|   (C12)
    if (g == G - 1 && tid == 0) L.ss[sys].edge[1] = fabs(Hs[2 * P + Wv].y);     // |b_{1,M}|
    if (service && lane == 0) {
        double* o = A.cta_out + (size_t)blockIdx.x * 8;
        o[0] = A_last; o[1] = B_last; o[2] = SV; o[3] = SC; o[4] = SS; o[5] = window;
    }
    // ---- one launch-wide synchronisation, then CTA 0 adds the slabs in a fixed order --------------------------
    const unsigned fin = (unsigned)(2 * n_steps) + 1u;
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
