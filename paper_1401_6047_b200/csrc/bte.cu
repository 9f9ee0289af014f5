// bte.cu -- host side of libbte_b200: the C ABI of include/bte.h.
// Product code: must not include, link or call anything under oracle/.
#include "../../include/bte.h"
#include "bte_internal.h"
#include "bte_sweep.cuh"
#include "bte_warpsweep.cuh"
#include "bte_resident.cuh"
#include "bte_pendulum.cuh"
#include "bte_lowprec.cuh"

#include <cmath>
#include <cstdarg>
#include <cstdio>
#include <cstring>
#include <algorithm>
#include <string>
#include <vector>

using namespace bte;

namespace {

thread_local std::string g_err;

// Every entry point runs on the device that owns the ctx's workspace, whatever device is current in the
// calling thread, and restores the caller's device on return.
struct DeviceGuard {
    int prev = -1;
    bool ok = true;
    explicit DeviceGuard(int dev) {
        int cur = -1;
        if (cudaGetDevice(&cur) != cudaSuccess) { ok = false; return; }
        if (cur != dev) {
            if (cudaSetDevice(dev) != cudaSuccess) { ok = false; return; }
            prev = cur;
        }
    }
    ~DeviceGuard() { if (prev >= 0) cudaSetDevice(prev); }
};
#define CTX_GUARD(c)                                                                                \
    DeviceGuard guard__((c)->device);                                                               \
    if (!guard__.ok) return fail(BTE_ECUDA, "cannot select CUDA device %d of this ctx", (c)->device)

int fail(int code, const char* fmt, ...) {
    char buf[512];
    va_list ap;
    va_start(ap, fmt);
    vsnprintf(buf, sizeof buf, fmt, ap);
    va_end(ap);
    g_err = buf;
    return code;
}

#define CUDA_TRY(expr)                                                                             \
    do {                                                                                           \
        cudaError_t e__ = (expr);                                                                  \
        if (e__ != cudaSuccess)                                                                    \
            return fail(BTE_ECUDA, "%s failed: %s (%s:%d)", #expr, cudaGetErrorString(e__),        \
                        __FILE__, __LINE__);                                                       \
    } while (0)

constexpr size_t ALIGN = 256;
size_t align_up(size_t x) { return (x + ALIGN - 1) / ALIGN * ALIGN; }

struct Offsets {
    int pitch;
    size_t state, state_bytes, cn, gm, phi, sc, ss, partial, gctl, rhalo, rout, rflag, total;
};

bool grid_ok(const bte_grid* g) {
    return g && g->n_harm >= 1 && g->n_phiy >= 3 && g->n_batch >= 1 && g->n_batch <= 65535 &&
           g->n_harm < 65535 && g->dt > 0.0 && std::isfinite(g->dt) && g->precision >= 0 && g->precision <= 2;
}

// resident (on-chip) variant: at most RES_MAX_CTAS slabs; usable shared memory per CTA (227 KB minus the
// kernel's static shared memory)
constexpr int RES_MAX_CTAS = 148;
constexpr size_t RES_SMEM_CAP = 227 * 1024 - 1024;
constexpr long long RES_BATCH_MAX_POINTS = 8192;   // automatic choice for batches: systems up to this many points

bool resident_possible(const bte_grid* g) {
    if (g->precision != 0) return false;                       // fp64 only
    // one system: up to RES_MAX_CTAS slabs (cooperative grid); a batch: one cluster of up to 16 CTAs per system
    const int gmax = g->n_batch == 1 ? RES_MAX_CTAS : 16;
    const int wc = (g->n_phiy + gmax - 1) / gmax;
    return resident_smem_bytes(g->n_harm, wc) <= RES_SMEM_CAP;
}

Offsets offsets_for(const bte_grid* g) {
    Offsets o{};
    o.pitch = (g->n_phiy + 7) / 8 * 8;
    const size_t rows = (size_t)g->n_harm + 1 + 2 * GHOST, nb = (size_t)g->n_batch, pitch = (size_t)o.pitch;
    size_t off = 0;
    const size_t elem = g->precision == 0 ? sizeof(double2) : sizeof(float2);   // fp32 storage: half the bytes
    o.state = off;   off = align_up(off + 2 * 2 * nb * rows * pitch * elem);
    o.state_bytes = 2 * 2 * nb * rows * pitch * elem;
    o.cn = off;      off = align_up(off + nb * rows * sizeof(double));
    o.gm = off;      off = align_up(off + nb * pitch * sizeof(double));
    o.phi = off;     off = align_up(off + nb * pitch * sizeof(double));
    o.sc = off;      off = align_up(off + nb * sizeof(SysConst));
    o.ss = off;      off = align_up(off + nb * sizeof(SysState));
    o.partial = off; off = align_up(off + (size_t)SWEEP_MAX_STEPS * nb * pitch * 2 * sizeof(double));
    o.gctl = off;    off = align_up(off + 64);
    // resident variant: edge columns of both grids of every slab, per-slab sums
    o.rhalo = off;
    if (resident_possible(g) && g->n_batch == 1)
        off = align_up(off + (size_t)2 * RES_MAX_HALO * 2 * RES_MAX_CTAS * 2 * (g->n_harm + 1) * sizeof(double2));
    o.rout = off;    off = align_up(off + std::max<size_t>(RES_MAX_CTAS, (size_t)g->n_batch * 16) * 8 * sizeof(double));
    o.rflag = off;   off = align_up(off + (size_t)RES_MAX_CTAS * sizeof(unsigned int));
    o.total = off;
    return o;
}

// I_n(x)/I_0(x), n = 0..N, by Miller's backward recurrence I_{n-1} = I_{n+1} + (2n/x) I_n (stable in this
// direction because I_n is the minimal solution); only ratios are needed, so no normalisation sum.
void bessel_i_ratios(double x, int N, std::vector<double>& r) {
    const int ns = N + 2 * (int)std::ceil(x) + 120;
    std::vector<double> t((size_t)ns + 2, 0.0);
    t[ns + 1] = 0.0;
    t[ns] = 1.0;
    for (int n = ns; n >= 1; --n) {
        t[n - 1] = t[n + 1] + (2.0 * n / x) * t[n];
        if (t[n - 1] > 1e200) {
            for (int j = n - 1; j <= ns; ++j) t[j] *= 1e-200;   // far tail underflows to 0, as it should
        }
    }
    r.resize((size_t)N + 1);
    for (int n = 0; n <= N; ++n) r[n] = t[n] / t[0];
}

enum Variant { VAR_AUTO = 0, VAR_SPLIT = 1, VAR_FUSED = 2, VAR_SWEEP = 3, VAR_RESIDENT = 4, VAR_WARPSWEEP = 5 };

}  // namespace

struct bte_ctx {
    bte_grid grid;
    std::vector<bte_params> params;
    Offsets off;
    char* ws;
    int device;             // ordinal of the device that owns the workspace
    cudaStream_t stream;
    Layout L;
    int64_t steps_issued;   // global step count requested so far (per-system count = min(this, budget))
    int64_t launches;
    // options
    int variant;
    int64_t graph_steps;    // -1 auto, 0 off
    int tile_rows;
    // fused (tile grid) launch plan
    int rows_per_chunk;
    dim3 fgrid;
    // sweep kernel (persistent, one wave, S steps per launch) launch plan
    bool has_budgets;
    int sweep_steps;                 // option: 0 = automatic, 1..SWEEP_MAX_STEPS
    int sweep_ctas;                  // option: grid-size override (0 = SMs x resident CTAs)
    int sweep_threads;               // option: 0 = automatic, 128, 256
    int sw_grid[SWEEP_MAX_STEPS + 1];   // grid of the S-step kernel; 0 = not usable for this problem
    int ws_grid[SWEEP_MAX_STEPS + 1];   // same for the warp kernel (bte_warpsweep.cuh), S = 2 .. WS_MAX_STEPS
    int sm_count;
    std::vector<int64_t> budgets;    // sorted distinct step budgets (n_steps_total > 0)
    std::vector<SysConst> sc_host;   // host copy of the per-system constants (re-uploaded by bte_set_steady_policy)
    bool steady_on;                  // steady-state detection / averaging policy in force
    // resident (on-chip) kernel launch plan
    int res_ctas_opt;                // option: slabs (0 = automatic)
    int res_mode;                    // -1 = not usable; 0 one CTA, 1 one cluster, 2 cooperative grid
    int res_G, res_Wc, res_T, res_HB;
    int res_halo_opt;                // option: halo columns of the grid mode (0 = automatic)
    size_t res_smem;
    // CUDA graph cache
    cudaGraph_t graph;
    cudaGraphExec_t graph_exec;
    int64_t graph_len;
    int graph_variant, graph_S;
};

namespace {

constexpr int FT = 128;   // threads per CTA of the fused kernel (strip of FT-2 = 126 columns)
constexpr int FD = 3;     // rows prefetched ahead

using FCfg = FusedCfg<FT, FD>;

int plan_fused(bte_ctx* c) {
    const int rows = c->grid.n_harm + 1;
    const int strips = (c->grid.n_phiy + FCfg::W - 1) / FCfg::W;
    int rpc = c->tile_rows;
    if (rpc <= 0) {
        // enough CTAs to fill 148 SMs several times over, but chunks long enough that the 2-row halo
        // recompute (and 6 extra row loads) per chunk stays at a few per cent
        const long long want = 148LL * 8;
        const long long have = (long long)strips * c->grid.n_batch;
        long long chunks = (want + have - 1) / have;
        if (chunks < 1) chunks = 1;
        rpc = (int)((rows + chunks - 1) / chunks);
        if (rpc < 32) rpc = 32;
    }
    if (rpc < 2) rpc = 2;
    if (rpc > rows) rpc = rows;
    if (rows >= 2 && rpc < 2) rpc = 2;
    c->rows_per_chunk = rpc;
    const int chunks = (rows + rpc - 1) / rpc;
    if (chunks > 65535) return fail(BTE_EINVAL, "too many row chunks");
    c->fgrid = dim3((unsigned)strips, (unsigned)chunks, (unsigned)c->grid.n_batch);
    return BTE_OK;
}

// ---- sweep kernel: S leap-frog steps per launch (bte_sweep.cuh) ----------------------------------------
// resident CTAs per SM the register budget of each instantiation is compiled for
template <int S> struct SweepMinB { static constexpr int v = S == 1 ? 4 : S == 2 ? 3 : 2; };

struct SweepFn { void* fn; size_t smem; int W; int T; int strips_per_band; };

// T = 128 threads per CTA (several CTAs per SM) or T = 256 (half the strip-halo overhead, longer DRAM bursts
// per row; S = 3 then runs one CTA per SM)
template <int T, int S>
SweepFn sweep_fn_ts(bool budgets) {
    using Cfg = SweepCfg<T, S>;
    constexpr int MB = T == 128 ? SweepMinB<S>::v : (S == 1 && T == 256 ? 2 : 1);
    return {budgets ? (void*)sweep_kernel<T, S, true, MB> : (void*)sweep_kernel<T, S, false, MB>,
            Cfg::smem_bytes, Cfg::W, T, 1};
}

SweepFn sweep_fn(int S, bool budgets, int wide) {
    if (wide == 2 && S == 1) return sweep_fn_ts<512, 1>(budgets);
    if (wide) {
        switch (S) {
            case 1: return sweep_fn_ts<256, 1>(budgets);
            case 2: return sweep_fn_ts<256, 2>(budgets);
            default: return sweep_fn_ts<256, 3>(budgets);
        }
    }
    switch (S) {
        case 1: return sweep_fn_ts<128, 1>(budgets);
        case 2: return sweep_fn_ts<128, 2>(budgets);
        default: return sweep_fn_ts<128, 3>(budgets);
    }
}
constexpr int RING_MAX_STEPS = 3;   // the shared-memory-ring kernel is instantiated for S = 1 .. 3
constexpr int WARP_MIN_ROWS = 32;   // automatic choice of the warp kernel: columns at least this long (config 3, 41 rows: 126 G against 105 G on the ring kernel)
constexpr int WARP_DEEP_ROWS = 320;  // automatic depth of the warp kernel: 4 steps per pass for columns at least this long
                                     // (x 32001 points, sustained G updates/s over 7200 steps at S = 3 / 4: 256 rows 158 / 154,
                                     // 288 rows 164 / 162, 320 rows 168 -> 160 / 167, 352 rows 170 -> 160 / 172,
                                     // 384 rows 172 -> 163 / 173, 513 rows 173 / 184, 1024 rows 181 / 191)
constexpr int WS_MAX_STEPS = 4;     // the register-resident kernel is instantiated for S = 2, 3, 4
static_assert(WS_MAX_STEPS <= SWEEP_MAX_STEPS, "partial sums are laid out for SWEEP_MAX_STEPS steps per pass");

// register-resident warp kernel (bte_warpsweep.cuh): S = 2, 3 steps per pass, K = BTE_WS_K columns per lane
constexpr int WS_K = BTE_WS_K;
// EB = bytes of a stored pair: 16 (fp64 state) or 8 (bte_grid.precision 1: fp32 storage, fp64 arithmetic)
template <int S, int EB>
SweepFn warpsweep_fn_s(bool budgets) {
    using Cfg = WarpCfg<S, WS_K, EB>;
    return {budgets ? (void*)warpsweep_kernel<S, WS_K, true, EB> : (void*)warpsweep_kernel<S, WS_K, false, EB>,
            Cfg::smem_bytes, Cfg::W, Cfg::T, Cfg::WARPS};
}
SweepFn warpsweep_fn(int S, bool budgets, int precision) {
    if (precision == 1)
        return S == 2 ? warpsweep_fn_s<2, 8>(budgets) : S == 3 ? warpsweep_fn_s<3, 8>(budgets) : warpsweep_fn_s<4, 8>(budgets);
    return S == 2 ? warpsweep_fn_s<2, 16>(budgets) : S == 3 ? warpsweep_fn_s<3, 16>(budgets) : warpsweep_fn_s<4, 16>(budgets);
}

// Wider CTAs pay off only for the HBM-bound one-step pass over long rows (4 or 8 KB DRAM bursts per row instead
// of 2 KB: 74 / 79 / 81 G updates/s on config 4 with 128 / 256 / 512 threads); the multi-step passes are faster
// with 128 (measured).  Returns 0 / 1 / 2 for 128 / 256 / 512 threads.
int sweep_wide(const bte_ctx* c, int S) {
    if (c->sweep_threads != 0) return c->sweep_threads == 512 ? 2 : c->sweep_threads == 256 ? 1 : 0;
    if (S != 1) return 0;
    return c->grid.n_phiy >= 8192 ? 2 : c->grid.n_phiy >= 4096 ? 1 : 0;
}

int plan_sweep(bte_ctx* c) {
    for (int S = 0; S <= SWEEP_MAX_STEPS; ++S) c->sw_grid[S] = c->ws_grid[S] = 0;
    if (c->grid.precision == 2) return BTE_OK;     // fp32 arithmetic: the split kernels only
    int dev = 0, sms = 0;
    CUDA_TRY(cudaGetDevice(&dev));
    CUDA_TRY(cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev));
    c->sm_count = sms;
    const long long rows_alloc = c->grid.n_harm + 1 + 2 * GHOST;
    // warp kernel: one CTA of WARPS independent warps per SM; a CTA range is counted in band-rows
    for (int S = 2; S <= WS_MAX_STEPS; ++S) {
        const SweepFn f = warpsweep_fn(S, c->has_budgets, c->grid.precision);
        int occ = 0;
        cudaError_t e = cudaFuncSetAttribute(f.fn, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)f.smem);
        if (e == cudaSuccess) e = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, f.fn, f.T, f.smem);
        if (e != cudaSuccess)
            return fail(BTE_ECUDA, "warpsweep_kernel<S=%d> setup failed: %s (is this an sm_100a device?)", S,
                        cudaGetErrorString(e));
        if (occ < 1) continue;
        const long long strips = (c->grid.n_phiy + f.W - 1) / f.W;
        const long long bands = (strips * c->grid.n_batch + f.strips_per_band - 1) / f.strips_per_band;
        const long long units = bands * (c->grid.n_harm + 1);
        if (2LL * c->grid.n_batch * rows_alloc * c->off.pitch >= (1LL << 31)) continue;   // 32-bit element offsets
        if (strips * (c->grid.n_harm + 1) >= (1LL << 31) || units >= (1LL << 31)) continue;
        long long g = (long long)sms * occ;
        // a segment costs about NS + HALO extra row iterations: a CTA should own a few times that many rows
        const long long min_rows = c->sweep_ctas > 0 ? 1 : 8 * S;
        if (c->sweep_ctas > 0) g = c->sweep_ctas;
        if (g > (units + min_rows - 1) / min_rows) g = (units + min_rows - 1) / min_rows;
        if (g < 1) g = 1;
        if (c->has_budgets && (long long)c->grid.n_batch / g + 2 > WarpCfg<2, WS_K>::MAX_SPAN) continue;
        c->ws_grid[S] = (int)g;
    }
    for (int S = 1; S <= RING_MAX_STEPS && c->grid.precision == 0; ++S) {
        c->sw_grid[S] = 0;
        const SweepFn f = sweep_fn(S, c->has_budgets, sweep_wide(c, S));
        int occ = 0;
        cudaError_t e = cudaFuncSetAttribute(f.fn, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)f.smem);
        if (e == cudaSuccess) e = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, f.fn, f.T, f.smem);
        if (e != cudaSuccess)
            return fail(BTE_ECUDA, "sweep_kernel<S=%d> setup failed: %s (is this an sm_100a device?)", S,
                        cudaGetErrorString(e));
        if (occ < 1) continue;
        const long long strips = (c->grid.n_phiy + f.W - 1) / f.W;
        const long long units = strips * (c->grid.n_harm + 1) * (long long)c->grid.n_batch;
        // 32-bit element offsets inside the kernel: both grids of one buffer, all systems
        if (2LL * c->grid.n_batch * rows_alloc * c->off.pitch >= (1LL << 31)) continue;
        if (units >= (1LL << 31)) continue;
        long long g = (long long)sms * occ;
        // a CTA should own enough rows to amortise the 3 NS - 1 fill/drain iterations of a segment
        const long long min_rows = c->sweep_ctas > 0 ? 1 : 8 * S;
        if (c->sweep_ctas > 0) g = c->sweep_ctas;
        if (g > (units + min_rows - 1) / min_rows) g = (units + min_rows - 1) / min_rows;
        if (g < 1) g = 1;
        // one CTA range may touch at most MAX_SPAN systems (shared-memory list)
        if (c->has_budgets && (long long)c->grid.n_batch / g + 2 > SweepCfg<FT, 1>::MAX_SPAN) continue;
        c->sw_grid[S] = (int)g;
    }
    return BTE_OK;
}

// ---- resident kernel: the whole time loop on chip (bte_resident.cuh) -------------------------------------
void* resident_fn(int mode) {
    return mode == 0 ? (void*)resident_kernel<0> : mode == 1 ? (void*)resident_kernel<1> : (void*)resident_kernel<2>;
}

// compute threads of a CTA (one more warp does the bookkeeping): one point per thread up to 31 warps
int resident_threads(int rows, int wc) {
    long long t = ((long long)rows * wc + 31) / 32 * 32;
    if (t > 992) t = 992;
    if (t < 64) t = 64;
    return (int)t;
}

// Try one (mode, G) combination: shared memory fits and the launch shape is schedulable.
bool resident_try(bte_ctx* c, int mode, int G) {
    const int M1 = c->grid.n_phiy, N = c->grid.n_harm;
    if (G < 1 || G > M1) return false;
    const int wc = (M1 + G - 1) / G;
    const int Ge = (M1 + wc - 1) / wc;          // slabs actually needed with this width
    if ((mode == 0) != (Ge == 1)) return false;
    if (mode == 1 && Ge != G) return false;    // cluster sizes are taken as given (2, 4, 8, 16)
    // grid mode: HB halo columns per side, one neighbour exchange per HB half-updates (bte_resident.cuh); every slab,
    // the last one included, must own at least HB columns
    int hb = 1;
    if (mode == 2) {
        hb = c->res_halo_opt > 0 ? c->res_halo_opt : 3;
        const int last = M1 - (Ge - 1) * wc;
        while (hb > 1 && (last < hb || resident_smem_bytes(N, wc, hb) > RES_SMEM_CAP)) --hb;
    }
    const size_t smem = resident_smem_bytes(N, wc, hb);
    if (smem > RES_SMEM_CAP) return false;
    void* fn = resident_fn(mode);
    const int T = resident_threads(N + 1, wc + 2 * (hb - 1));
    if (cudaFuncSetAttribute(fn, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem) != cudaSuccess) {
        cudaGetLastError();
        return false;
    }
    if (mode == 1) {
        if (Ge > 8 && cudaFuncSetAttribute(fn, cudaFuncAttributeNonPortableClusterSizeAllowed, 1) != cudaSuccess) {
            cudaGetLastError();
            return false;
        }
        cudaLaunchConfig_t cfg{};
        cfg.gridDim = dim3(Ge); cfg.blockDim = dim3(T + 32); cfg.dynamicSmemBytes = smem; cfg.stream = c->stream;
        cudaLaunchAttribute at[1];
        at[0].id = cudaLaunchAttributeClusterDimension;
        at[0].val.clusterDim.x = Ge; at[0].val.clusterDim.y = 1; at[0].val.clusterDim.z = 1;
        cfg.attrs = at; cfg.numAttrs = 1;
        int nclusters = 0;
        if (cudaOccupancyMaxActiveClusters(&nclusters, fn, &cfg) != cudaSuccess || nclusters < 1) {
            cudaGetLastError();
            return false;
        }
    } else if (mode == 2) {
        int occ = 0, coop = 0, dev = 0;
        cudaGetDevice(&dev);
        cudaDeviceGetAttribute(&coop, cudaDevAttrCooperativeLaunch, dev);
        if (!coop || cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, fn, T + 32, smem) != cudaSuccess ||
            (long long)occ * c->sm_count < Ge) {
            cudaGetLastError();
            return false;
        }
    }
    c->res_mode = mode; c->res_G = Ge; c->res_Wc = wc; c->res_T = T; c->res_smem = smem; c->res_HB = hb;
    return true;
}

int plan_resident(bte_ctx* c) {
    c->res_mode = -1;
    if (!resident_possible(&c->grid)) return BTE_OK;
    const long long pts = (long long)(c->grid.n_harm + 1) * c->grid.n_phiy;
    const int maxg = c->sm_count < RES_MAX_CTAS ? c->sm_count : RES_MAX_CTAS;
    if (c->res_ctas_opt > 0) {                  // explicit slab count: 1 = one CTA, 2..16 = cluster, more = grid
        const int G = c->res_ctas_opt;
        if (G == 1) resident_try(c, 0, 1);
        else if (G <= 16 && resident_try(c, 1, G)) {}
        else if (G <= maxg && c->grid.n_batch == 1) resident_try(c, 2, G);
        return BTE_OK;
    }
    // automatic: the fewest slabs that leave at most 512 points per CTA (one point per thread, the SM's fp64 and
    // shared-memory pipes far from saturated; measured on config 0: 3.4 / 1.9 / 1.7 us per step with 4 / 8 / 16
    // CTAs); synchronisation cost grows with the number of CTAs: __syncthreads < cluster barrier < neighbour
    // flags through L2
    if (pts <= 512 && resident_try(c, 0, 1)) return BTE_OK;
    // one system of more than 16 x 512 points: cooperative grid with 3 halo columns per side (one neighbour exchange per
    // 3 half-updates), as many slabs as leave about one point per thread and half-update (measured: config 1 5.5 us per
    // step on a cluster of 16, 3.5 us on a grid of 67; config 2 9.0 -> 7.1 us on 148 slabs)
    if (c->grid.n_batch == 1 && pts > 16 * 512) {
        const int hb = c->res_halo_opt > 0 ? c->res_halo_opt : 3;
        const int rows = c->grid.n_harm + 1;
        int own = 992 / rows - 2 * (hb - 1);
        if (own < hb) own = hb;
        int G = (c->grid.n_phiy + own - 1) / own;
        if (G > maxg) G = maxg;
        if (G > 16 && resident_try(c, 2, G)) return BTE_OK;
    }
    for (int G = 2; G <= 16; G *= 2)
        if ((pts / G <= 512 || G == 16) && resident_try(c, 1, G)) return BTE_OK;
    for (int G = 8; G >= 2; G /= 2)             // 16 not schedulable / does not fit: smaller clusters that fit
        if (resident_try(c, 1, G)) return BTE_OK;
    if (resident_try(c, 0, 1)) return BTE_OK;
    if (c->grid.n_batch == 1) resident_try(c, 2, maxg);    // the grid mode synchronises CTAs of ONE system
    return BTE_OK;
}

int launch_resident(bte_ctx* c, int64_t n_steps) {
    ResidentArgs A{};
    A.G = c->res_G; A.Wc = c->res_Wc; A.T = c->res_T; A.n_steps = n_steps; A.HB = c->res_HB;
    A.halo = (double2*)(c->ws + c->off.rhalo);
    A.cta_out = (double*)(c->ws + c->off.rout);
    A.flag = (unsigned int*)(c->ws + c->off.rflag);
    void* fn = resident_fn(c->res_mode);
    void* args[] = {&c->L, &A};
    cudaLaunchConfig_t cfg{};
    cfg.gridDim = dim3((unsigned)c->res_G * (unsigned)c->grid.n_batch);   // one CTA / cluster per system
    cfg.blockDim = dim3(c->res_T + 32); cfg.dynamicSmemBytes = c->res_smem;
    cfg.stream = c->stream;
    cudaLaunchAttribute at[1];
    cfg.attrs = at; cfg.numAttrs = 0;
    if (c->res_mode == 1) {
        at[0].id = cudaLaunchAttributeClusterDimension;
        at[0].val.clusterDim.x = c->res_G; at[0].val.clusterDim.y = 1; at[0].val.clusterDim.z = 1;
        cfg.numAttrs = 1;
    } else if (c->res_mode == 2) {
        CUDA_TRY(cudaMemsetAsync(A.flag, 0, (size_t)c->res_G * sizeof(unsigned int), c->stream));
        at[0].id = cudaLaunchAttributeCooperative;
        at[0].val.cooperative = 1;
        cfg.numAttrs = 1;
    }
    CUDA_TRY(cudaLaunchKernelExC(&cfg, fn, args));
    c->launches += 1;
    return BTE_OK;
}

int effective_variant(const bte_ctx* c) {
    if (c->grid.precision == 2) return VAR_SPLIT;
    if (c->grid.precision == 1) {
        // fp32 storage: multi-step passes through the warp kernel (half the HBM bytes), single steps (remainders, budget
        // cuts) through the two-launch form
        const bool ok = c->ws_grid[3] > 0 && c->grid.n_harm + 1 >= WARP_MIN_ROWS;
        return ok && (c->variant == VAR_AUTO || c->variant == VAR_WARPSWEEP || c->variant == VAR_RESIDENT) ? VAR_WARPSWEEP
                                                                                                         : VAR_SPLIT;
    }
    // one-step launches of the warp kernel's plan run the ring kernel (the HBM-bound form), so both must be usable
    const bool warp_ok = c->sw_grid[1] > 0 && c->ws_grid[2] > 0;
    if (c->variant == VAR_WARPSWEEP && warp_ok) return VAR_WARPSWEEP;
    // AUTO, and what runs when the resident kernel is not used: a streaming kernel.  Long columns: the warp kernel
    // (registers + tensor memory; a segment costs about 2 NS extra row iterations, so it wants a long march over n); short
    // columns (batches of small systems): the shared-memory-ring kernel at S = 2.
    const bool streaming = c->variant == VAR_AUTO || c->variant == VAR_RESIDENT || c->variant == VAR_WARPSWEEP;
    if (streaming && warp_ok && c->ws_grid[3] > 0 && c->grid.n_harm + 1 >= WARP_MIN_ROWS) return VAR_WARPSWEEP;
    if (streaming || c->variant == VAR_SWEEP) return c->sw_grid[1] > 0 ? VAR_SWEEP : VAR_FUSED;
    return c->variant;
}

bool is_sweep(int var) { return var == VAR_SWEEP || var == VAR_WARPSWEEP; }

// is an s-step launch available in the effective streaming variant?  (one-step launches always run the
// shared-memory-ring kernel: the HBM-bound form, bte_sweep.cuh)
bool sweep_has(const bte_ctx* c, int var, int s) {
    if (s == 1) return c->grid.precision == 0 ? c->sw_grid[1] > 0 : true;   // fp32 storage: the two-launch form
    return var == VAR_WARPSWEEP ? c->ws_grid[s] > 0 : (s <= RING_MAX_STEPS && c->sw_grid[s] > 0);
}

// steps fused per launch by the sweep kernels (the other variants advance one step per launch group)
int sweep_steps(const bte_ctx* c) {
    const int var = effective_variant(c);
    if (!is_sweep(var)) return 1;
    int S;
    if (var == VAR_WARPSWEEP) {
        // 4 steps per pass on long columns: 16 B of HBM traffic per update.  Alone it is 2 % slower than 3 (184 against
        // 188 G on config 4: 14 of 96 columns per strip are halos instead of 10), but the 3-step pass loses its clocks under
        // sustained load (172-175 G after ~0.2 s) and the 4-step pass does not (183-184.6 G
        // throughout); shorter columns run too slowly to lose their clocks and pay more for the deeper pipeline
        S = c->sweep_steps > 0 ? c->sweep_steps : (c->grid.n_harm + 1 >= WARP_DEEP_ROWS ? 4 : 3);
    } else {
        // ring kernel: 3 steps per pass when the march over n is long enough to amortise the 3 NS - 1
        // fill/drain iterations of a segment, else 2 (measured on configs 3 and 4)
        S = c->sweep_steps > 0 ? c->sweep_steps : (c->grid.n_harm + 1 >= 96 ? 3 : 2);
    }
    while (S > 1 && !sweep_has(c, var, S)) --S;
    return S;
}

// kernel, launch shape and grid of an s-step launch of the effective streaming variant
SweepFn sweep_launch(const bte_ctx* c, int var, int s, int* grid) {
    if (var == VAR_WARPSWEEP && s >= 2) {
        *grid = c->ws_grid[s];
        return warpsweep_fn(s, c->has_budgets, c->grid.precision);
    }
    *grid = c->sw_grid[s];
    return sweep_fn(s, c->has_budgets, sweep_wide(c, s));
}

void drop_graph(bte_ctx* c) {
    if (c->graph_exec) cudaGraphExecDestroy(c->graph_exec);
    if (c->graph) cudaGraphDestroy(c->graph);
    c->graph_exec = nullptr;
    c->graph = nullptr;
    c->graph_len = 0;
}

dim3 split_grid(const bte_ctx* c) {
    return dim3((unsigned)((c->grid.n_phiy + 127) / 128), (unsigned)(c->grid.n_harm + 1),
                (unsigned)c->grid.n_batch);
}

// column chunks x systems of reduce_finalize_kernel (each chunk at least one block's worth of columns)
dim3 reduce_grid(const bte_ctx* c) {
    int nb = (c->grid.n_phiy + 255) / 256;
    if (nb > RED_BLOCKS) nb = RED_BLOCKS;
    return dim3((unsigned)nb, (unsigned)c->grid.n_batch);
}

int launches_per_step(const bte_ctx* c) { return effective_variant(c) == VAR_SPLIT ? 3 : 1; }

// Issue one launch group with plain launches: S steps (sweep kernel) or one step (other variants).
int launch_steps(bte_ctx* c, int S) {
    const int var = effective_variant(c);
    const bool single32 = c->grid.precision != 0 && S == 1;   // fp32 storage: single steps in the two-launch form
    if (is_sweep(var) && !single32) {
        int grid = 0;
        const SweepFn f = sweep_launch(c, var, S, &grid);
        void* args[] = {&c->L};
        CUDA_TRY(cudaLaunchKernel(f.fn, dim3(grid), dim3(f.T), args, f.smem, c->stream));
    } else if (var == VAR_FUSED) {
        fused_step_kernel<FT, FD><<<c->fgrid, FT, FCfg::smem_bytes, c->stream>>>(c->L, c->rows_per_chunk);
    } else {
        const dim3 g = split_grid(c);
        if (c->grid.precision == 0) {
            half_update_kernel<<<g, 128, 0, c->stream>>>(c->L, 0);
            half_update_kernel<<<g, 128, 0, c->stream>>>(c->L, 1);
            reduce_finalize_kernel<double2><<<reduce_grid(c), 256, 0, c->stream>>>(c->L, 1);
        } else if (c->grid.precision == 1) {
            half_update32_kernel<1><<<g, 128, 0, c->stream>>>(c->L, 0);
            half_update32_kernel<1><<<g, 128, 0, c->stream>>>(c->L, 1);
            reduce_finalize_kernel<float2><<<reduce_grid(c), 256, 0, c->stream>>>(c->L, 1);
        } else {
            half_update32_kernel<2><<<g, 128, 0, c->stream>>>(c->L, 0);
            half_update32_kernel<2><<<g, 128, 0, c->stream>>>(c->L, 1);
            reduce_finalize_kernel<float2><<<reduce_grid(c), 256, 0, c->stream>>>(c->L, 1);
        }
    }
    CUDA_TRY(cudaGetLastError());
    c->launches += single32 ? 3 : launches_per_step(c);
    return BTE_OK;
}

// Build a graph of `len` launch groups (each S steps) from explicit kernel nodes (no stream capture: safe
// with any caller stream).  Kernels take no per-step argument -- the step counter lives on the device -- so
// one graph can be replayed any number of times.
int build_graph(bte_ctx* c, int64_t len, int S) {
    drop_graph(c);
    CUDA_TRY(cudaGraphCreate(&c->graph, 0));
    cudaGraphNode_t prev = nullptr;
    const int var = effective_variant(c);
    int mode0 = 0, mode1 = 1, adv = 1;
    int rpc = c->rows_per_chunk;
    for (int64_t s = 0; s < len; ++s) {
        auto add = [&](void* fn, dim3 grid, dim3 block, size_t smem, void** args) -> cudaError_t {
            cudaKernelNodeParams p{};
            p.func = fn; p.gridDim = grid; p.blockDim = block; p.sharedMemBytes = (unsigned)smem;
            p.kernelParams = args; p.extra = nullptr;
            cudaGraphNode_t node;
            cudaError_t e = cudaGraphAddKernelNode(&node, c->graph, prev ? &prev : nullptr, prev ? 1 : 0, &p);
            prev = node;
            return e;
        };
        if (is_sweep(var)) {
            int grid = 0;
            const SweepFn f = sweep_launch(c, var, S, &grid);
            void* args[] = {&c->L};
            CUDA_TRY(add(f.fn, dim3(grid), dim3(f.T), f.smem, args));
        } else if (var == VAR_FUSED) {
            void* args[] = {&c->L, &rpc};
            CUDA_TRY(add((void*)fused_step_kernel<FT, FD>, c->fgrid, dim3(FT), FCfg::smem_bytes, args));
        } else {
            const dim3 g = split_grid(c);
            void* a0[] = {&c->L, &mode0};
            void* a1[] = {&c->L, &mode1};
            void* a2[] = {&c->L, &adv};
            void* hu = c->grid.precision == 0 ? (void*)half_update_kernel
                       : c->grid.precision == 1 ? (void*)half_update32_kernel<1> : (void*)half_update32_kernel<2>;
            void* rf = c->grid.precision == 0 ? (void*)reduce_finalize_kernel<double2> : (void*)reduce_finalize_kernel<float2>;
            CUDA_TRY(add(hu, g, dim3(128), 0, a0));
            CUDA_TRY(add(hu, g, dim3(128), 0, a1));
            CUDA_TRY(add(rf, reduce_grid(c), dim3(256), 0, a2));
        }
    }
    CUDA_TRY(cudaGraphInstantiate(&c->graph_exec, c->graph, 0));
    c->graph_len = len;
    c->graph_variant = var;
    c->graph_S = S;
    return BTE_OK;
}

int64_t auto_graph_steps(const bte_ctx* c) {
    // a step of a small grid takes a few microseconds: launch overhead dominates => replay graphs
    const double pts = (double)(c->grid.n_harm + 1) * c->grid.n_phiy * c->grid.n_batch;
    if (pts > 4.0e6) return 0;
    return 64;
}

// steps until the next step budget strictly after global step k (INT64_MAX if none)
int64_t steps_to_next_budget(const bte_ctx* c, int64_t k) {
    auto it = std::upper_bound(c->budgets.begin(), c->budgets.end(), k);
    return it == c->budgets.end() ? INT64_MAX : *it - k;
}

// which ping-pong buffer holds the current state of a system (device-side flag; synchronises the stream)
int live_buffer(bte_ctx* c, int sys, int* buf) {
    SysState st;
    CUDA_TRY(cudaMemcpyAsync(&st, c->ws + c->off.ss + (size_t)sys * sizeof(SysState), sizeof(SysState),
                             cudaMemcpyDeviceToHost, c->stream));
    CUDA_TRY(cudaStreamSynchronize(c->stream));
    *buf = st.buf & 1;
    return BTE_OK;
}

}  // namespace

// shared with the other translation units of the library (bte_internal.h); hidden visibility
void bte_internal_set_error(const char* text) { g_err = text ? text : ""; }

extern "C" {

const char* bte_last_error(void) { return g_err.c_str(); }


size_t bte_workspace_bytes(const bte_grid* grid) {
    if (!grid_ok(grid)) return 0;
    return offsets_for(grid).total;
}

int bte_create(const bte_grid* grid, const bte_params* params, void* workspace, size_t bytes,
               void* cuda_stream, bte_ctx** out) {
    if (out) *out = nullptr;
    if (!out || !grid || !params || !workspace) return fail(BTE_EINVAL, "bte_create: NULL argument");
    if (!grid_ok(grid))
        return fail(BTE_EINVAL, "bte_create: need n_harm >= 1, n_phiy >= 3, 1 <= n_batch <= 65535, dt > 0, precision 0..2");
    const Offsets off = offsets_for(grid);
    if (((long long)grid->n_harm + 1 + 2 * GHOST) * off.pitch >= (1LL << 31) - 8LL * off.pitch)
        return fail(BTE_EINVAL, "bte_create: (n_harm+1) * n_phiy must stay below 2^31 points per system");
    if (bytes < off.total) return fail(BTE_ENOMEM, "bte_create: workspace has %zu bytes, %zu needed", bytes, off.total);
    if (((uintptr_t)workspace % ALIGN) != 0) return fail(BTE_ENOMEM, "bte_create: workspace must be 256-byte aligned");
    const int N = grid->n_harm, M1 = grid->n_phiy, M = M1 - 1, nb = grid->n_batch;
    for (int s = 0; s < nb; ++s) {
        const bte_params& p = params[s];
        const bool finite = std::isfinite(p.E_dc) && std::isfinite(p.E_omega) && std::isfinite(p.omega) &&
                            std::isfinite(p.B) && std::isfinite(p.mu) && std::isfinite(p.alpha) &&
                            std::isfinite(p.phiy_min) && std::isfinite(p.phiy_max) && std::isfinite(p.kappa_scale);
        if (!finite || !(p.mu > 0.0) || !(p.alpha > 0.0) || !(p.phiy_max > p.phiy_min) ||
            p.n_steps_total < 0 || p.avg_start_step < 0)
            return fail(BTE_EINVAL, "bte_create: system %d: need finite parameters, mu > 0, alpha > 0, phiy_max > phiy_min", s);
        const double dphi = (p.phiy_max - p.phiy_min) / M;
        if (std::fabs(p.B) * grid->dt / dphi >= 2.0)
            return fail(BTE_EUNSTABLE, "bte_create: system %d: |B| dt / dphi = %g >= 2 (scheme unstable)", s,
                        std::fabs(p.B) * grid->dt / dphi);
    }
    cudaStream_t stream = (cudaStream_t)cuda_stream;
    // the device that owns the workspace is the device of this ctx (first CUDA call: after all argument checks)
    int device = 0;
    {
        cudaPointerAttributes attr{};
        if (cudaPointerGetAttributes(&attr, workspace) != cudaSuccess || attr.type != cudaMemoryTypeDevice) {
            cudaGetLastError();
            return fail(BTE_EINVAL, "bte_create: workspace is not a device pointer");
        }
        device = attr.device;
    }
    DeviceGuard guard__(device);
    if (!guard__.ok) return fail(BTE_ECUDA, "bte_create: cannot select CUDA device %d", device);

    // host tables: phi_y lattice (C8), Gaussian factor and c_n of eq. (15)-(16) (C1, C13)
    const size_t rows = (size_t)N + 1 + 2 * GHOST, pitch = (size_t)off.pitch;   // with ghost entries (zero)
    std::vector<double> cn(nb * rows, 0.0), gm(nb * pitch, 0.0), phi(nb * pitch, 0.0), ratios;
    std::vector<SysConst> sc((size_t)nb);
    const double PI = 3.14159265358979323846;
    for (int s = 0; s < nb; ++s) {
        const bte_params& p = params[s];
        const double dphi = (p.phiy_max - p.phiy_min) / M;
        const double centre = 0.5 * (p.phiy_min + p.phiy_max);
        for (int m = 0; m < M1; ++m) {
            const double ph = centre + (m - M / 2.0) * dphi;
            double g = std::exp(-p.mu * ph * ph / 2.0);
            if (g < 1e-300) g = 0.0;   // input-recipe clamp (C19)
            phi[s * pitch + m] = ph;
            gm[s * pitch + m] = g;
        }
        bessel_i_ratios(p.mu, N, ratios);
        const double pref = std::sqrt(p.mu / (2.0 * PI * p.alpha));
        cn[s * rows + GHOST] = (1.0 / (2.0 * PI)) * pref;
        for (int n = 1; n <= N; ++n) cn[s * rows + GHOST + n] = (ratios[n] / PI) * pref;
        SysConst& k = sc[s];
        k.E_dc = p.E_dc; k.E_omega = p.E_omega; k.omega = p.omega; k.B = p.B; k.dphi = dphi;
        k.kappa_dt = p.kappa_scale * p.B * grid->dt / (4.0 * dphi);
        k.norm_scale = 2.0 * PI * std::sqrt(p.alpha) * dphi;
        k.v_scale = PI * std::sqrt(p.alpha) * dphi;
        k.n_steps_total = p.n_steps_total; k.avg_start_step = p.avg_start_step;
        k.period_steps = 0; k.window_steps = 0; k.steady_tol = 0.0; k.n_avg_periods = 0; k.min_relax_periods = 0;
    }
    char* ws = (char*)workspace;
    CUDA_TRY(cudaMemcpyAsync(ws + off.cn, cn.data(), cn.size() * sizeof(double), cudaMemcpyHostToDevice, stream));
    CUDA_TRY(cudaMemcpyAsync(ws + off.gm, gm.data(), gm.size() * sizeof(double), cudaMemcpyHostToDevice, stream));
    CUDA_TRY(cudaMemcpyAsync(ws + off.phi, phi.data(), phi.size() * sizeof(double), cudaMemcpyHostToDevice, stream));
    CUDA_TRY(cudaMemcpyAsync(ws + off.sc, sc.data(), sc.size() * sizeof(SysConst), cudaMemcpyHostToDevice, stream));
    CUDA_TRY(cudaMemsetAsync(ws + off.state, 0, off.state_bytes, stream));   // ghost rows stay zero forever
    CUDA_TRY(cudaMemsetAsync(ws + off.ss, 0, (size_t)nb * sizeof(SysState), stream));
    CUDA_TRY(cudaMemsetAsync(ws + off.partial, 0, (size_t)SWEEP_MAX_STEPS * nb * pitch * 2 * sizeof(double), stream));
    CUDA_TRY(cudaMemsetAsync(ws + off.gctl, 0, 64, stream));
    CUDA_TRY(cudaStreamSynchronize(stream));   // host tables go out of scope

    bte_ctx* c = new bte_ctx();
    c->grid = *grid;
    c->params.assign(params, params + nb);
    c->off = off; c->ws = ws; c->stream = stream; c->device = device;
    c->L.N = N; c->L.M1 = M1; c->L.pitch = off.pitch; c->L.n_batch = nb; c->L.dt = grid->dt;
    c->L.nu = 1.0 + 0.5 * grid->dt; c->L.xi = 1.0 - 0.5 * grid->dt; c->L.nu2 = c->L.nu * c->L.nu;
    c->L.hd = 0.5 * grid->dt;
    c->L.state = (double2*)(ws + off.state);
    c->L.cn = (const double*)(ws + off.cn);
    c->L.gm = (const double*)(ws + off.gm);
    c->L.phi = (const double*)(ws + off.phi);
    c->L.sc = (const SysConst*)(ws + off.sc);
    c->L.ss = (SysState*)(ws + off.ss);
    c->L.partial = (double*)(ws + off.partial);
    c->L.gctl = (unsigned int*)(ws + off.gctl);
    c->has_budgets = false;
    c->sc_host = sc; c->steady_on = false;
    for (int s = 0; s < nb; ++s) c->has_budgets = c->has_budgets || params[s].n_steps_total > 0;
    for (int s = 0; s < nb; ++s)
        if (params[s].n_steps_total > 0) c->budgets.push_back(params[s].n_steps_total);
    std::sort(c->budgets.begin(), c->budgets.end());
    c->budgets.erase(std::unique(c->budgets.begin(), c->budgets.end()), c->budgets.end());
    c->sweep_steps = 0; c->sweep_ctas = 0; c->sm_count = 0; c->graph_S = 0; c->sweep_threads = 0;
    c->res_ctas_opt = 0; c->res_mode = -1; c->res_G = 0; c->res_Wc = 0; c->res_T = 0; c->res_smem = 0;
    c->res_HB = 1; c->res_halo_opt = 0;
    for (int S = 0; S <= SWEEP_MAX_STEPS; ++S) c->sw_grid[S] = c->ws_grid[S] = 0;
    c->steps_issued = 0; c->launches = 0;
    c->variant = VAR_AUTO; c->graph_steps = -1;
    c->tile_rows = 0;
    c->graph = nullptr; c->graph_exec = nullptr; c->graph_len = 0; c->graph_variant = 0;
    int rc = plan_fused(c);
    if (rc != BTE_OK) { delete c; return rc; }
    cudaError_t e = cudaFuncSetAttribute(fused_step_kernel<FT, FD>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                         (int)FCfg::smem_bytes);
    if (e != cudaSuccess) {
        delete c;
        return fail(BTE_ECUDA, "cudaFuncSetAttribute failed: %s (is this an sm_100a device?)", cudaGetErrorString(e));
    }
    rc = plan_sweep(c);
    if (rc != BTE_OK) { delete c; return rc; }
    rc = plan_resident(c);
    if (rc != BTE_OK) { delete c; return rc; }
    *out = c;
    return BTE_OK;
}

int bte_init_equilibrium(bte_ctx* c) {
    if (!c) return fail(BTE_EINVAL, "bte_init_equilibrium: NULL ctx");
    CTX_GUARD(c);
    const dim3 g((unsigned)((c->off.pitch + 127) / 128), (unsigned)(c->grid.n_harm + 1), (unsigned)c->grid.n_batch);
    if (c->grid.precision == 0) {
        init_state_kernel<<<g, 128, 0, c->stream>>>(c->L);
        half_update_kernel<<<split_grid(c), 128, 0, c->stream>>>(c->L, 2);   // start-up z^{1/2}, L202
        reduce_finalize_kernel<double2><<<reduce_grid(c), 256, 0, c->stream>>>(c->L, 0);
    } else {
        init_state32_kernel<<<g, 128, 0, c->stream>>>(c->L, c->grid.precision);
        if (c->grid.precision == 1) half_update32_kernel<1><<<split_grid(c), 128, 0, c->stream>>>(c->L, 2);
        else half_update32_kernel<2><<<split_grid(c), 128, 0, c->stream>>>(c->L, 2);
        reduce_finalize_kernel<float2><<<reduce_grid(c), 256, 0, c->stream>>>(c->L, 0);
    }
    CUDA_TRY(cudaGetLastError());
    c->launches += 3;
    c->steps_issued = 0;
    return BTE_OK;
}

int bte_step(bte_ctx* c, int64_t n_steps) {
    if (!c) return fail(BTE_EINVAL, "bte_step: NULL ctx");
    if (n_steps < 0) return fail(BTE_EINVAL, "bte_step: n_steps < 0");
    CTX_GUARD(c);
    int64_t left = n_steps;
    // lattices that fit on chip: ONE launch runs the whole time loop out of shared memory (automatic choice
    // from 4 steps on -- below that the load/store of the state is not amortised)
    // (batches: only small systems -- a batch of mid-size systems streams faster through the sweep kernel)
    const bool res_auto = c->variant == VAR_AUTO && n_steps >= 4 &&
                          (c->grid.n_batch == 1 || (long long)(c->grid.n_harm + 1) * c->grid.n_phiy <= RES_BATCH_MAX_POINTS);
    if (c->res_mode >= 0 && (c->variant == VAR_RESIDENT || res_auto) && !c->steady_on) {
        int64_t n = n_steps;
        if (c->grid.n_batch == 1) {            // (a batch: the kernel ends every system at its own budget)
            const int64_t tot = c->params[0].n_steps_total;
            if (tot > 0) n = std::min<int64_t>(n, std::max<int64_t>(0, tot - c->steps_issued));
        }
        while (n > 0) {                      // 32-bit half-update counters inside the kernel: <= 2^30 steps a launch
            const int64_t m = std::min<int64_t>(n, (int64_t)1 << 30);
            const int rc = launch_resident(c, m);
            if (rc != BTE_OK) return rc;
            n -= m;
        }
        c->steps_issued += n_steps;
        return BTE_OK;
    }
    const int S = sweep_steps(c);
    const int var = effective_variant(c);
    // launch-bound grids: replay a graph of glen launch groups of S steps each (not with step budgets:
    // a budget boundary inside a group changes the group)
    const int64_t glen = c->has_budgets ? 0 : (c->graph_steps < 0 ? auto_graph_steps(c) : c->graph_steps);
    if (glen > 1 && left >= glen * S) {
        if (!c->graph_exec || c->graph_len != glen || c->graph_variant != var || c->graph_S != S) {
            int rc = build_graph(c, glen, S);
            if (rc != BTE_OK) return rc;
        }
        while (left >= glen * S) {
            CUDA_TRY(cudaGraphLaunch(c->graph_exec, c->stream));
            c->launches += glen * launches_per_step(c);
            left -= glen * S;
            c->steps_issued += glen * S;
        }
    }
    // every system has a budget and all of them are spent: nothing left to launch
    bool all_budgeted = c->has_budgets;
    for (size_t i = 0; all_budgeted && i < c->params.size(); ++i) all_budgeted = c->params[i].n_steps_total > 0;
    while (left > 0) {
        if (all_budgeted && c->steps_issued >= c->budgets.back()) {
            c->steps_issued += left;
            break;
        }
        // an s-step launch must not contain a budget boundary in its interior (a system that would freeze
        // after fewer than s steps): shorten the group to end exactly on the next boundary
        int64_t s = std::min<int64_t>(S, left);
        if (c->has_budgets) s = std::min<int64_t>(s, steps_to_next_budget(c, c->steps_issued));
        while (s > 1 && is_sweep(var) && !sweep_has(c, var, (int)s)) --s;
        int rc = launch_steps(c, (int)s);
        if (rc != BTE_OK) return rc;
        left -= s;
        c->steps_issued += s;
    }
    return BTE_OK;
}

int bte_observables(bte_ctx* c, bte_obs* out) {
    if (!c || !out) return fail(BTE_EINVAL, "bte_observables: NULL argument");
    CTX_GUARD(c);
    std::vector<SysState> ss((size_t)c->grid.n_batch);
    CUDA_TRY(cudaMemcpyAsync(ss.data(), c->ws + c->off.ss, ss.size() * sizeof(SysState), cudaMemcpyDeviceToHost, c->stream));
    CUDA_TRY(cudaStreamSynchronize(c->stream));
    for (int s = 0; s < c->grid.n_batch; ++s) {
        bte_obs& o = out[s];
        o.step = ss[s].k; o.t = (double)ss[s].k * c->grid.dt; o.norm = ss[s].norm; o.v_dr = ss[s].v_dr;
        o.sum_v_dt = ss[s].sum_v; o.sum_vcos_dt = ss[s].sum_c; o.sum_vsin_dt = ss[s].sum_s;
        o.window = ss[s].window; o.edge_leak = ss[s].edge_leak;
    }
    return BTE_OK;
}

int bte_destroy(bte_ctx* c) {
    if (!c) return BTE_OK;
    DeviceGuard guard__(c->device);
    drop_graph(c);
    delete c;
    return BTE_OK;
}

// element offset (in lattice points) of row 0 of one (buffer, grid, system) array inside the state region
size_t state_offset(const bte_ctx* c, int buf, int grid_id, int system) {
    const size_t gp = (size_t)(c->grid.n_harm + 1 + 2 * GHOST) * c->off.pitch;
    return (((size_t)buf * 2 + grid_id) * c->grid.n_batch + system) * gp + (size_t)GHOST * c->off.pitch;
}

int bte_get_state(bte_ctx* c, int32_t system, int32_t grid_id, double* a, double* b) {
    if (!c || !a || !b) return fail(BTE_EINVAL, "bte_get_state: NULL argument");
    if (system < 0 || system >= c->grid.n_batch || grid_id < 0 || grid_id > 1)
        return fail(BTE_EINVAL, "bte_get_state: bad system or grid index");
    CTX_GUARD(c);
    const int rows = c->grid.n_harm + 1, M1 = c->grid.n_phiy, pitch = c->off.pitch;
    int buf = 0;
    { const int rc = live_buffer(c, system, &buf); if (rc != BTE_OK) return rc; }
    const size_t cnt = (size_t)rows * M1;
    const dim3 g((unsigned)((M1 + 255) / 256), (unsigned)rows);
    double *stage_a, *stage_b;
    // rows 0..N of the other buffer of this system are dead between steps: they serve as staging
    if (c->grid.precision == 0) {
        const double2* z = c->L.state + state_offset(c, buf, grid_id, system);
        stage_a = (double*)(c->L.state + state_offset(c, buf ^ 1, grid_id, system));
        stage_b = stage_a + cnt;
        deinterleave_kernel<<<g, 256, 0, c->stream>>>(z, stage_a, stage_b, rows, M1, pitch);
    } else {   // fp32 arrays hold 8 B per point: a is staged in the dead whole-grid array, b in the fractional one
        const float2* z = (const float2*)c->L.state + state_offset(c, buf, grid_id, system);
        stage_a = (double*)((float2*)c->L.state + state_offset(c, buf ^ 1, 0, system));
        stage_b = (double*)((float2*)c->L.state + state_offset(c, buf ^ 1, 1, system));
        deinterleave32_kernel<<<g, 256, 0, c->stream>>>(z, stage_a, stage_b, rows, M1, pitch);
    }
    CUDA_TRY(cudaGetLastError());
    c->launches += 1;
    CUDA_TRY(cudaMemcpyAsync(a, stage_a, cnt * sizeof(double), cudaMemcpyDeviceToHost, c->stream));
    CUDA_TRY(cudaMemcpyAsync(b, stage_b, cnt * sizeof(double), cudaMemcpyDeviceToHost, c->stream));
    CUDA_TRY(cudaStreamSynchronize(c->stream));
    return BTE_OK;
}

int bte_set_state(bte_ctx* c, int32_t system, int32_t grid_id, const double* a, const double* b) {
    if (!c || !a || !b) return fail(BTE_EINVAL, "bte_set_state: NULL argument");
    if (system < 0 || system >= c->grid.n_batch || grid_id < 0 || grid_id > 1)
        return fail(BTE_EINVAL, "bte_set_state: bad system or grid index");
    CTX_GUARD(c);
    const int rows = c->grid.n_harm + 1, M1 = c->grid.n_phiy, pitch = c->off.pitch;
    int buf = 0;
    { const int rc = live_buffer(c, system, &buf); if (rc != BTE_OK) return rc; }
    const size_t cnt = (size_t)rows * M1;
    const dim3 g((unsigned)((pitch + 255) / 256), (unsigned)rows);
    if (c->grid.precision == 0) {
        double2* z = c->L.state + state_offset(c, buf, grid_id, system);
        double* stage = (double*)(c->L.state + state_offset(c, buf ^ 1, grid_id, system));
        CUDA_TRY(cudaMemcpyAsync(stage, a, cnt * sizeof(double), cudaMemcpyHostToDevice, c->stream));
        CUDA_TRY(cudaMemcpyAsync(stage + cnt, b, cnt * sizeof(double), cudaMemcpyHostToDevice, c->stream));
        interleave_kernel<<<g, 256, 0, c->stream>>>(z, stage, stage + cnt, rows, M1, pitch);
    } else {
        float2* z = (float2*)c->L.state + state_offset(c, buf, grid_id, system);
        double* stage_a = (double*)((float2*)c->L.state + state_offset(c, buf ^ 1, 0, system));
        double* stage_b = (double*)((float2*)c->L.state + state_offset(c, buf ^ 1, 1, system));
        CUDA_TRY(cudaMemcpyAsync(stage_a, a, cnt * sizeof(double), cudaMemcpyHostToDevice, c->stream));
        CUDA_TRY(cudaMemcpyAsync(stage_b, b, cnt * sizeof(double), cudaMemcpyHostToDevice, c->stream));
        interleave32_kernel<<<g, 256, 0, c->stream>>>(z, stage_a, stage_b, rows, M1, pitch);
    }
    c->launches += 1;
    if (grid_id == 0) {   // keep norm / v_dr of the observables consistent with the new whole grid
        // the reduction reads the live buffer of every system; harmless for the others
        if (c->grid.precision == 0) reduce_finalize_kernel<double2><<<reduce_grid(c), 256, 0, c->stream>>>(c->L, 0);
        else reduce_finalize_kernel<float2><<<reduce_grid(c), 256, 0, c->stream>>>(c->L, 0);
        c->launches += 1;
    }
    CUDA_TRY(cudaGetLastError());
    CUDA_TRY(cudaStreamSynchronize(c->stream));
    return BTE_OK;
}

// ---- state exchange for the whole batch (one launch group, one synchronisation) -----------------------------
namespace {
// every system's live state into buffer 0 (systems whose flag says 1 are copied, then the flags are cleared), so
// that the host knows where everything is without reading the flags back
int normalise_buffers(bte_ctx* c) {
    const size_t per = (size_t)(c->grid.n_harm + 1 + 2 * GHOST) * c->off.pitch;
    const dim3 g((unsigned)std::min<size_t>((per + 255) / 256, 4096), 2, (unsigned)c->grid.n_batch);
    if (c->grid.precision == 0) copy_live_to_buffer0_kernel<double2><<<g, 256, 0, c->stream>>>(c->L);
    else copy_live_to_buffer0_kernel<float2><<<g, 256, 0, c->stream>>>(c->L);
    clear_buffer_flags_kernel<<<(c->grid.n_batch + 255) / 256, 256, 0, c->stream>>>(c->L);
    CUDA_TRY(cudaGetLastError());
    c->launches += 2;
    return BTE_OK;
}
}  // namespace

int bte_get_state_batch(bte_ctx* c, int32_t grid_id, double* a, double* b) {
    if (!c || !a || !b) return fail(BTE_EINVAL, "bte_get_state_batch: NULL argument");
    if (grid_id < 0 || grid_id > 1) return fail(BTE_EINVAL, "bte_get_state_batch: bad grid index");
    CTX_GUARD(c);
    const int rows = c->grid.n_harm + 1, M1 = c->grid.n_phiy, nb = c->grid.n_batch;
    const size_t cnt = (size_t)rows * M1;
    if (c->grid.precision != 0) {                      // fp32 storage: system by system (reference-grade variants)
        for (int s = 0; s < nb; ++s) {
            const int rc = bte_get_state(c, s, grid_id, a + (size_t)s * cnt, b + (size_t)s * cnt);
            if (rc != BTE_OK) return rc;
        }
        return BTE_OK;
    }
    { const int rc = normalise_buffers(c); if (rc != BTE_OK) return rc; }
    // de-interleave every system from buffer 0 into its own rows 0..N of buffer 1 (dead between steps)
    const dim3 g((unsigned)((M1 + 255) / 256), (unsigned)rows, (unsigned)nb);
    deinterleave_batch_kernel<<<g, 256, 0, c->stream>>>(c->L, grid_id);
    CUDA_TRY(cudaGetLastError());
    c->launches += 1;
    const size_t gp = (size_t)(rows + 2 * GHOST) * c->off.pitch * sizeof(double2);   // bytes between systems
    const double* stage = (const double*)(c->L.state + state_offset(c, 1, grid_id, 0));
    CUDA_TRY(cudaMemcpy2DAsync(a, cnt * sizeof(double), stage, gp, cnt * sizeof(double), (size_t)nb,
                               cudaMemcpyDeviceToHost, c->stream));
    CUDA_TRY(cudaMemcpy2DAsync(b, cnt * sizeof(double), stage + cnt, gp, cnt * sizeof(double), (size_t)nb,
                               cudaMemcpyDeviceToHost, c->stream));
    CUDA_TRY(cudaStreamSynchronize(c->stream));
    return BTE_OK;
}

int bte_set_state_batch(bte_ctx* c, int32_t grid_id, const double* a, const double* b) {
    if (!c || !a || !b) return fail(BTE_EINVAL, "bte_set_state_batch: NULL argument");
    if (grid_id < 0 || grid_id > 1) return fail(BTE_EINVAL, "bte_set_state_batch: bad grid index");
    CTX_GUARD(c);
    const int rows = c->grid.n_harm + 1, M1 = c->grid.n_phiy, nb = c->grid.n_batch;
    const size_t cnt = (size_t)rows * M1;
    if (c->grid.precision != 0) {
        for (int s = 0; s < nb; ++s) {
            const int rc = bte_set_state(c, s, grid_id, a + (size_t)s * cnt, b + (size_t)s * cnt);
            if (rc != BTE_OK) return rc;
        }
        return BTE_OK;
    }
    { const int rc = normalise_buffers(c); if (rc != BTE_OK) return rc; }
    const size_t gp = (size_t)(rows + 2 * GHOST) * c->off.pitch * sizeof(double2);
    double* stage = (double*)(c->L.state + state_offset(c, 1, grid_id, 0));
    CUDA_TRY(cudaMemcpy2DAsync(stage, gp, a, cnt * sizeof(double), cnt * sizeof(double), (size_t)nb,
                               cudaMemcpyHostToDevice, c->stream));
    CUDA_TRY(cudaMemcpy2DAsync(stage + cnt, gp, b, cnt * sizeof(double), cnt * sizeof(double), (size_t)nb,
                               cudaMemcpyHostToDevice, c->stream));
    const dim3 g((unsigned)((c->off.pitch + 255) / 256), (unsigned)rows, (unsigned)nb);
    interleave_batch_kernel<<<g, 256, 0, c->stream>>>(c->L, grid_id);
    c->launches += 1;
    if (grid_id == 0) {   // keep norm / v_dr of the observables consistent with the new whole grids
        reduce_finalize_kernel<double2><<<reduce_grid(c), 256, 0, c->stream>>>(c->L, 0);
        c->launches += 1;
    }
    CUDA_TRY(cudaGetLastError());
    CUDA_TRY(cudaStreamSynchronize(c->stream));
    return BTE_OK;
}

int bte_set_steady_policy(bte_ctx* c, double rel_tol, int32_t n_avg_periods, int32_t min_relax_periods) {
    if (!c) return fail(BTE_EINVAL, "bte_set_steady_policy: NULL context");
    CTX_GUARD(c);
    if (!(rel_tol >= 0.0) || !std::isfinite(rel_tol) || (rel_tol > 0.0 && (n_avg_periods < 1 || min_relax_periods < 0)))
        return fail(BTE_EINVAL, "bte_set_steady_policy: need rel_tol >= 0, n_avg_periods >= 1, min_relax_periods >= 0");
    if (rel_tol > 0.0) {
        const int var = effective_variant(c);
        if (c->grid.precision != 0 || !is_sweep(var))
            return fail(BTE_EINVAL, "bte_set_steady_policy: runs in the streaming sweep kernels only (fp64, variant 0, 3 or 5)");
    }
    const double PI = 3.14159265358979323846;
    for (size_t s = 0; s < c->sc_host.size(); ++s) {
        SysConst& k = c->sc_host[s];
        const double w = std::fabs(c->params[s].omega);
        // comparison interval: one ac period; a dc system (omega = 0): one relaxation time (C23)
        const double P = w > 0.0 ? 2.0 * PI / (w * c->grid.dt) : 1.0 / c->grid.dt;
        k.period_steps = std::max<long long>(1, std::llround(P));
        k.window_steps = std::max<long long>(1, std::llround((double)n_avg_periods * P));
        k.steady_tol = rel_tol; k.n_avg_periods = n_avg_periods; k.min_relax_periods = min_relax_periods;
    }
    CUDA_TRY(cudaMemcpyAsync(c->ws + c->off.sc, c->sc_host.data(), c->sc_host.size() * sizeof(SysConst),
                             cudaMemcpyHostToDevice, c->stream));
    CUDA_TRY(cudaStreamSynchronize(c->stream));
    const bool was = c->has_budgets;
    c->steady_on = rel_tol > 0.0;
    // finished systems are compacted out of the launches like systems past their budget
    c->has_budgets = c->steady_on;
    for (size_t s = 0; s < c->params.size(); ++s) c->has_budgets = c->has_budgets || c->params[s].n_steps_total > 0;
    if (was != c->has_budgets) { drop_graph(c); return plan_sweep(c); }
    return BTE_OK;
}

int bte_steady_info(bte_ctx* c, int64_t* steady_step, int32_t* phase) {
    if (!c || !steady_step || !phase) return fail(BTE_EINVAL, "bte_steady_info: NULL argument");
    CTX_GUARD(c);
    std::vector<SysState> ss((size_t)c->grid.n_batch);
    CUDA_TRY(cudaMemcpyAsync(ss.data(), c->ws + c->off.ss, ss.size() * sizeof(SysState), cudaMemcpyDeviceToHost, c->stream));
    CUDA_TRY(cudaStreamSynchronize(c->stream));
    for (int s = 0; s < c->grid.n_batch; ++s) { steady_step[s] = ss[s].steady_step; phase[s] = ss[s].phase; }
    return BTE_OK;
}

int bte_get_option(bte_ctx* c, const char* key, int64_t* out) {
    if (!c || !key || !out) return fail(BTE_EINVAL, "bte_get_option: NULL argument");
    if (!strcmp(key, "effective_variant")) { *out = effective_variant(c); return BTE_OK; }
    if (!strcmp(key, "effective_sweep_steps")) { *out = sweep_steps(c); return BTE_OK; }
    if (!strcmp(key, "resident_usable")) { *out = c->res_mode >= 0 ? 1 : 0; return BTE_OK; }
    if (!strcmp(key, "resident_ctas")) { *out = c->res_mode >= 0 ? c->res_G : 0; return BTE_OK; }
    if (!strcmp(key, "device")) { *out = c->device; return BTE_OK; }
    if (!strcmp(key, "variant")) { *out = c->variant; return BTE_OK; }
    return fail(BTE_EINVAL, "bte_get_option: unknown key '%s'", key);
}

int bte_reconstruct_pdf(bte_ctx* c, int32_t system, int32_t grid_id, int32_t n_phix, double* f) {
    if (!c || !f) return fail(BTE_EINVAL, "bte_reconstruct_pdf: NULL argument");
    if (system < 0 || system >= c->grid.n_batch || grid_id < 0 || grid_id > 1)
        return fail(BTE_EINVAL, "bte_reconstruct_pdf: bad system or grid index");
    if (n_phix < 1 || n_phix > 2048) return fail(BTE_EINVAL, "bte_reconstruct_pdf: n_phix must be in [1, 2048]");
    if (c->grid.precision != 0) return fail(BTE_EINVAL, "bte_reconstruct_pdf: fp64 contexts only");
    CTX_GUARD(c);
    const int rows = c->grid.n_harm + 1, M1 = c->grid.n_phiy, pitch = c->off.pitch;
    int buf = 0;
    { const int rc = live_buffer(c, system, &buf); if (rc != BTE_OK) return rc; }
    const size_t gp = (size_t)(rows + 2 * GHOST) * pitch, row0 = (size_t)GHOST * pitch;
    const double2* z = c->L.state + (((size_t)buf * 2 + grid_id) * c->grid.n_batch + system) * gp + row0;
    constexpr int KT = 16;
    const dim3 g((unsigned)((M1 + 127) / 128), (unsigned)((n_phix + KT - 1) / KT));
    pdf_kernel<KT><<<g, 128, 2 * (size_t)n_phix * sizeof(double), c->stream>>>(z, f, rows, M1, pitch, n_phix);
    CUDA_TRY(cudaGetLastError());
    c->launches += 1;
    return BTE_OK;
}

size_t bte_pendulum_workspace_bytes(int32_t n) {
    return n < 1 ? 0 : (size_t)n * (sizeof(PendulumParams) + sizeof(PendulumOut));
}

int bte_pendulum_averages(const bte_pendulum_params* params, int32_t n, int32_t n_phase, double h, int32_t n_rk,
                          void* workspace, size_t bytes, void* cuda_stream, bte_pendulum_out* out) {
    static_assert(sizeof(bte_pendulum_params) == sizeof(PendulumParams) && sizeof(bte_pendulum_out) == sizeof(PendulumOut),
                  "ABI structs mirror the device structs");
    if (!params || !out || !workspace) return fail(BTE_EINVAL, "bte_pendulum_averages: NULL argument");
    if (n < 1 || n > 65535 || n_phase < 1 || n_rk < 2 || (n_rk & 1) || !(h > 0.0) || !std::isfinite(h))
        return fail(BTE_EINVAL, "bte_pendulum_averages: need 1 <= n <= 65535, n_phase >= 1, even n_rk >= 2, h > 0");
    for (int i = 0; i < n; ++i)
        if (!std::isfinite(params[i].E_dc) || !std::isfinite(params[i].E_omega) || !std::isfinite(params[i].omega) ||
            !std::isfinite(params[i].B))
            return fail(BTE_EINVAL, "bte_pendulum_averages: parameter set %d is not finite", i);
    if (bytes < bte_pendulum_workspace_bytes(n)) return fail(BTE_ENOMEM, "bte_pendulum_averages: workspace too small");
    cudaStream_t stream = (cudaStream_t)cuda_stream;
    PendulumParams* dp = (PendulumParams*)workspace;
    PendulumOut* dout = (PendulumOut*)((char*)workspace + (size_t)n * sizeof(PendulumParams));
    CUDA_TRY(cudaMemcpyAsync(dp, params, (size_t)n * sizeof(PendulumParams), cudaMemcpyHostToDevice, stream));
    pendulum_kernel<<<n, 128, 0, stream>>>(dp, dout, n_phase, h, n_rk);
    CUDA_TRY(cudaGetLastError());
    CUDA_TRY(cudaMemcpyAsync(out, dout, (size_t)n * sizeof(PendulumOut), cudaMemcpyDeviceToHost, stream));
    CUDA_TRY(cudaStreamSynchronize(stream));
    return BTE_OK;
}

int bte_set_option(bte_ctx* c, const char* key, int64_t value) {
    if (!c || !key) return fail(BTE_EINVAL, "bte_set_option: NULL argument");
    CTX_GUARD(c);
    if (!strcmp(key, "variant")) {
        if (value < 0 || value > 5) return fail(BTE_EINVAL, "variant must be 0, 1, 2, 3, 4 or 5");
        c->variant = (int)value;
        drop_graph(c);
        return BTE_OK;
    }
    if (!strcmp(key, "graph_steps")) {
        if (value < -1 || value > 4096) return fail(BTE_EINVAL, "graph_steps must be in [-1, 4096]");
        c->graph_steps = value;
        return BTE_OK;
    }
    if (!strcmp(key, "tile_rows")) {
        if (value < 0 || (value > 0 && value < 2)) return fail(BTE_EINVAL, "tile_rows must be 0 or >= 2");
        c->tile_rows = (int)value;
        drop_graph(c);
        return plan_fused(c);
    }
    if (!strcmp(key, "sweep_ctas")) {   // CTAs of the persistent sweep kernel (0 = SMs x occupancy)
        if (value < 0 || value > 65535) return fail(BTE_EINVAL, "%s must be in [0, 65535]", key);
        c->sweep_ctas = (int)value;
        drop_graph(c);
        return plan_sweep(c);
    }
    if (!strcmp(key, "resident_ctas")) {   // slabs of the resident kernel: 1 = one CTA, 2..16 = cluster, more = grid
        if (value < 0 || value > RES_MAX_CTAS) return fail(BTE_EINVAL, "resident_ctas must be in [0, %d]", RES_MAX_CTAS);
        c->res_ctas_opt = (int)value;
        return plan_resident(c);
    }
    if (!strcmp(key, "resident_halo")) {   // halo columns per side of the resident kernel's grid mode (0 = automatic)
        if (value < 0 || value > RES_MAX_HALO) return fail(BTE_EINVAL, "resident_halo must be in [0, %d]", RES_MAX_HALO);
        c->res_halo_opt = (int)value;
        return plan_resident(c);
    }
    if (!strcmp(key, "sweep_threads")) {   // threads per CTA of the sweep kernel: 128 or 256 (0 = automatic)
        if (value != 0 && value != 128 && value != 256 && value != 512)
            return fail(BTE_EINVAL, "sweep_threads must be 0, 128, 256 or 512 (512: one-step pass only)");
        c->sweep_threads = (int)value;
        drop_graph(c);
        return plan_sweep(c);
    }
    if (!strcmp(key, "sweep_steps")) {   // leap-frog steps fused per launch of the sweep kernel (0 = automatic)
        if (value < 0 || value > SWEEP_MAX_STEPS) return fail(BTE_EINVAL, "sweep_steps must be in [0, %d]", SWEEP_MAX_STEPS);
        c->sweep_steps = (int)value;
        drop_graph(c);
        return BTE_OK;
    }
    return fail(BTE_EINVAL, "bte_set_option: unknown key '%s'", key);
}

int bte_launch_count(bte_ctx* c, int64_t* out) {
    if (!c || !out) return fail(BTE_EINVAL, "bte_launch_count: NULL argument");
    *out = c->launches;
    return BTE_OK;
}

}  // extern "C"
