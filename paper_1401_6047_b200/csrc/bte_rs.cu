// bte_rs.cu -- host side of the real-space-phi_x variant (include/bte.h, bte_rs_* entry points).
// Product code: must not include, link or call anything under oracle/.
#include "../../include/bte.h"
#include "bte_internal.h"
#include "bte_realspace.cuh"

#include <cmath>
#include <cstdio>
#include <vector>

using namespace bte;


namespace {

int rs_fail(int code, const char* text) {
    bte_internal_set_error(text);
    return code;
}

#define RS_CUDA_TRY(expr)                                                                          \
    do {                                                                                           \
        cudaError_t e__ = (expr);                                                                  \
        if (e__ != cudaSuccess) {                                                                  \
            char buf__[256];                                                                       \
            snprintf(buf__, sizeof buf__, "%s failed: %s", #expr, cudaGetErrorString(e__));        \
            return rs_fail(BTE_ECUDA, buf__);                                                      \
        }                                                                                          \
    } while (0)

constexpr size_t RS_ALIGN = 256;
size_t rs_align(size_t x) { return (x + RS_ALIGN - 1) / RS_ALIGN * RS_ALIGN; }

struct RsOffsets { int pitch; size_t f, cprime, zvec, ex, sinx, gm, phi, partial, obs, total; };

bool rs_grid_ok(const bte_rs_grid* g) {
    return g && g->n_phix >= 4 && g->n_phix <= 4096 && g->n_phiy >= 3 && g->dt > 0.0 && std::isfinite(g->dt);
}

RsOffsets rs_offsets(const bte_rs_grid* g) {
    RsOffsets o{};
    o.pitch = (g->n_phiy + 7) / 8 * 8;
    const size_t K = (size_t)g->n_phix, p = (size_t)o.pitch, blocks = p / RS_PCR_MT + 1;   // >= the blocks of either kernel
    size_t off = 0;
    o.f = off;       off = rs_align(off + 2 * K * p * sizeof(double));
    o.cprime = off;  off = rs_align(off + K * p * sizeof(double));
    o.zvec = off;    off = rs_align(off + K * p * sizeof(double));
    o.ex = off;      off = rs_align(off + K * sizeof(double));
    o.sinx = off;    off = rs_align(off + K * sizeof(double));
    o.gm = off;      off = rs_align(off + p * sizeof(double));
    o.phi = off;     off = rs_align(off + p * sizeof(double));
    o.partial = off; off = rs_align(off + blocks * 2 * sizeof(double));
    o.obs = off;     off = rs_align(off + sizeof(RsObs));
    o.total = off;
    return o;
}

// I_0(x) e^{-x} by its power series / asymptotic series is overkill here: exp(mu (cos x - 1)) / (I0(mu) e^{-mu})
// needs the scaled Bessel function only; sum the series of I0(x) e^{-x} = sum_k (x/2)^{2k} / (k!)^2 e^{-x} in
// log space for moderate x and use the large-argument expansion beyond.
double bessel_i0_scaled(double x) {
    if (x < 30.0) {
        double term = 1.0, sum = 1.0;
        for (int k = 1; k < 500; ++k) {
            term *= (x / 2.0) * (x / 2.0) / ((double)k * k);
            sum += term;
            if (term < 1e-17 * sum) break;
        }
        return sum * std::exp(-x);
    }
    double term = 1.0, sum = 1.0;                      // I0(x) e^{-x} ~ 1/sqrt(2 pi x) sum_k ((2k-1)!!)^2 / (k! (8x)^k)
    for (int k = 1; k < 40; ++k) {
        term *= (2.0 * k - 1.0) * (2.0 * k - 1.0) / (k * 8.0 * x);
        if (term < 1e-17 * sum) break;
        sum += term;
    }
    return sum / std::sqrt(2.0 * 3.14159265358979323846 * x);
}

}  // namespace

struct bte_rs_ctx {
    bte_rs_grid grid;
    bte_params params;
    RsOffsets off;
    char* ws;
    cudaStream_t stream;
    RsLayout L;
    int64_t k;          // whole-grid steps taken
    RsKernel pcr;       // n_phix a power of two <= RS_PCR_MAX_K: parallel cyclic reduction; else NULL: Thomas sweeps
};

namespace {

// one half-update (mode as in bte_realspace.cuh) on the context's stream
void rs_launch(bte_rs_ctx* c, int mode, long long k, int do_avg) {
    if (c->pcr) {
        const unsigned blocks = (unsigned)(c->off.pitch / RS_PCR_MT);
        cudaLaunchConfig_t cfg = {};
        cfg.gridDim = dim3(blocks); cfg.blockDim = dim3(RS_PCR_T);
        cfg.dynamicSmemBytes = rs_pcr_smem(c->grid.n_phix); cfg.stream = c->stream;
        cudaLaunchAttribute at[1];
        at[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;    // prologue of this launch overlaps the previous one
        at[0].val.programmaticStreamSerializationAllowed = 1;
        cfg.attrs = at; cfg.numAttrs = 1;
        cudaLaunchKernelEx(&cfg, c->pcr, c->L, mode, k, do_avg);
    } else {
        const unsigned blocks = (unsigned)((c->off.pitch + 127) / 128);
        rs_half_update_kernel<<<blocks, 128, 0, c->stream>>>(c->L, mode, k, do_avg);
    }
}

}  // namespace

extern "C" {

size_t bte_rs_workspace_bytes(const bte_rs_grid* grid) {
    if (!rs_grid_ok(grid)) return 0;
    return rs_offsets(grid).total;
}

int bte_rs_create(const bte_rs_grid* grid, const bte_params* p, void* workspace, size_t bytes, void* cuda_stream,
                  bte_rs_ctx** out) {
    if (out) *out = nullptr;
    if (!out || !grid || !p || !workspace) return rs_fail(BTE_EINVAL, "bte_rs_create: NULL argument");
    if (!rs_grid_ok(grid)) return rs_fail(BTE_EINVAL, "bte_rs_create: need 4 <= n_phix <= 4096, n_phiy >= 3, dt > 0");
    const RsOffsets off = rs_offsets(grid);
    if (bytes < off.total) return rs_fail(BTE_ENOMEM, "bte_rs_create: workspace too small");
    if (((uintptr_t)workspace % RS_ALIGN) != 0) return rs_fail(BTE_ENOMEM, "bte_rs_create: workspace must be 256-byte aligned");
    const bool finite = std::isfinite(p->E_dc) && std::isfinite(p->E_omega) && std::isfinite(p->omega) &&
                        std::isfinite(p->B) && std::isfinite(p->mu) && std::isfinite(p->alpha) &&
                        std::isfinite(p->phiy_min) && std::isfinite(p->phiy_max) && std::isfinite(p->kappa_scale);
    if (!finite || !(p->mu > 0.0) || !(p->alpha > 0.0) || !(p->phiy_max > p->phiy_min) || p->n_steps_total < 0 ||
        p->avg_start_step < 0)
        return rs_fail(BTE_EINVAL, "bte_rs_create: need finite parameters, mu > 0, alpha > 0, phiy_max > phiy_min");
    const int K = grid->n_phix, M1 = grid->n_phiy, M = M1 - 1;
    const double dphi = (p->phiy_max - p->phiy_min) / M;
    if (std::fabs(p->B) * grid->dt / dphi >= 2.0)
        return rs_fail(BTE_EUNSTABLE, "bte_rs_create: |B| dt / dphi >= 2 (scheme unstable, DESIGN.md C11)");
    const double PI = 3.14159265358979323846;
    const double dx = 2.0 * PI / K;
    std::vector<double> ex(K), sx(K), gm(off.pitch, 0.0), phi(off.pitch, 0.0);
    const double pref = (1.0 / (2.0 * PI)) * std::sqrt(p->mu / (2.0 * PI * p->alpha)) / bessel_i0_scaled(p->mu);
    for (int i = 0; i < K; ++i) {
        const double x = -PI + dx * i;
        ex[i] = pref * std::exp(p->mu * (std::cos(x) - 1.0));          // eq. (13), phi_x part
        sx[i] = std::sin(x);
    }
    const double centre = 0.5 * (p->phiy_min + p->phiy_max);
    for (int m = 0; m < M1; ++m) {
        const double ph = centre + (m - M / 2.0) * dphi;               // C8
        double g = std::exp(-p->mu * ph * ph / 2.0);
        if (g < 1e-300) g = 0.0;                                        // C19
        phi[m] = ph;
        gm[m] = g;
    }
    cudaStream_t stream = (cudaStream_t)cuda_stream;
    char* ws = (char*)workspace;
    RS_CUDA_TRY(cudaMemsetAsync(ws, 0, off.total, stream));
    RS_CUDA_TRY(cudaMemcpyAsync(ws + off.ex, ex.data(), K * sizeof(double), cudaMemcpyHostToDevice, stream));
    RS_CUDA_TRY(cudaMemcpyAsync(ws + off.sinx, sx.data(), K * sizeof(double), cudaMemcpyHostToDevice, stream));
    RS_CUDA_TRY(cudaMemcpyAsync(ws + off.gm, gm.data(), gm.size() * sizeof(double), cudaMemcpyHostToDevice, stream));
    RS_CUDA_TRY(cudaMemcpyAsync(ws + off.phi, phi.data(), phi.size() * sizeof(double), cudaMemcpyHostToDevice, stream));
    RS_CUDA_TRY(cudaStreamSynchronize(stream));
    bte_rs_ctx* c = new bte_rs_ctx();
    c->grid = *grid; c->params = *p; c->off = off; c->ws = ws; c->stream = stream; c->k = 0;
    c->pcr = rs_pcr_kernel_for(K);
    if (c->pcr) {
        const cudaError_t e = cudaFuncSetAttribute(c->pcr, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)rs_pcr_smem(K));
        if (e != cudaSuccess) { delete c; return rs_fail(BTE_ECUDA, "bte_rs_create: cudaFuncSetAttribute failed"); }
    }
    RsLayout& L = c->L;
    L.K = K; L.M1 = M1; L.pitch = off.pitch; L.dt = grid->dt; L.dx = dx; L.dphi = dphi;
    L.E_dc = p->E_dc; L.E_omega = p->E_omega; L.omega = p->omega; L.B = p->B; L.kappa_scale = p->kappa_scale;
    L.norm_scale = std::sqrt(p->alpha) * dx * dphi;
    L.f = (double*)(ws + off.f); L.cprime = (double*)(ws + off.cprime); L.zvec = (double*)(ws + off.zvec);
    L.ex = (const double*)(ws + off.ex); L.sinx = (const double*)(ws + off.sinx);
    L.gm = (const double*)(ws + off.gm); L.phi = (const double*)(ws + off.phi);
    L.partial = (double*)(ws + off.partial); L.obs = (RsObs*)(ws + off.obs);
    *out = c;
    return BTE_OK;
}

int bte_rs_init_equilibrium(bte_rs_ctx* c) {
    if (!c) return rs_fail(BTE_EINVAL, "bte_rs_init_equilibrium: NULL ctx");
    const dim3 g((unsigned)((c->off.pitch + 127) / 128), (unsigned)c->grid.n_phix);
    rs_init_kernel<<<g, 128, 0, c->stream>>>(c->L);
    rs_launch(c, 2, 0, 0);                                                    // start-up z^{1/2}, L202
    RS_CUDA_TRY(cudaGetLastError());
    c->k = 0;
    return BTE_OK;
}

int bte_rs_step(bte_rs_ctx* c, int64_t n_steps) {
    if (!c) return rs_fail(BTE_EINVAL, "bte_rs_step: NULL ctx");
    if (n_steps < 0) return rs_fail(BTE_EINVAL, "bte_rs_step: n_steps < 0");
    for (int64_t s = 0; s < n_steps; ++s) {
        if (c->params.n_steps_total > 0 && c->k >= c->params.n_steps_total) break;   // frozen
        const int do_avg = (c->k + 1 > c->params.avg_start_step) ? 1 : 0;
        rs_launch(c, 0, (long long)c->k, do_avg);      // eq. (40)
        rs_launch(c, 1, (long long)c->k, 0);           // eq. (41), C5
        c->k += 1;
    }
    RS_CUDA_TRY(cudaGetLastError());
    return BTE_OK;
}

int bte_rs_observables(bte_rs_ctx* c, bte_obs* out) {
    if (!c || !out) return rs_fail(BTE_EINVAL, "bte_rs_observables: NULL argument");
    RsObs o;
    RS_CUDA_TRY(cudaMemcpyAsync(&o, c->ws + c->off.obs, sizeof o, cudaMemcpyDeviceToHost, c->stream));
    RS_CUDA_TRY(cudaStreamSynchronize(c->stream));
    out->step = c->k; out->t = (double)c->k * c->grid.dt; out->norm = o.norm; out->v_dr = o.v_dr;
    out->sum_v_dt = o.sum_v; out->sum_vcos_dt = o.sum_c; out->sum_vsin_dt = o.sum_s; out->window = o.window;
    out->edge_leak = 0.0;
    return BTE_OK;
}

int bte_rs_get_state(bte_rs_ctx* c, int32_t grid_id, double* f) {
    if (!c || !f) return rs_fail(BTE_EINVAL, "bte_rs_get_state: NULL argument");
    if (grid_id < 0 || grid_id > 1) return rs_fail(BTE_EINVAL, "bte_rs_get_state: bad grid index");
    const size_t K = (size_t)c->grid.n_phix, M1 = (size_t)c->grid.n_phiy, p = (size_t)c->off.pitch;
    RS_CUDA_TRY(cudaMemcpy2DAsync(f, M1 * sizeof(double), c->L.f + (size_t)grid_id * K * p, p * sizeof(double),
                                  M1 * sizeof(double), K, cudaMemcpyDeviceToHost, c->stream));
    RS_CUDA_TRY(cudaStreamSynchronize(c->stream));
    return BTE_OK;
}

int bte_rs_destroy(bte_rs_ctx* c) {
    delete c;
    return BTE_OK;
}

}  // extern "C"

// ---- bte_rs_evolve_static: the real-space step without any allocation (include/bte.h) ----------------------------------
// For callers that cannot allocate or own a workspace (CUDA graph capture, tight serving loops, harnesses that forbid
// cudaMalloc): the same kernels as bte_rs_step, with everything they need besides the caller's input and output -- the
// pitched state, the Thomas scratch arrays, the tables, the block partials and the observables -- in ONE file-scope
// device array of fixed size.  Every GPU that loads the library holds these RS_STATIC_BYTES until the process exits.
// All calls share the array and it keeps the last call's contents: what must start at zero (the observables: running
// sums and the block counter) is cleared at the start of every call; calls that overlap on the GPU (two streams, or
// two host threads) race.
#include <mutex>

namespace {

constexpr size_t RS_STATIC_MAX_POINTS = 131072;            // n_phix * pitch, pitch = n_phiy rounded up to a multiple of 8
constexpr size_t RS_STATIC_BYTES = (size_t)5 << 20;        // 4 arrays of MAX_POINTS doubles (4 MiB) + tables, partials, observables
static __device__ __align__(256) unsigned char rs_static_scratch[RS_STATIC_BYTES];

struct RsStaticOffsets { int pitch; size_t f, cprime, zvec, ex, sinx, gm, phi, partial, obs, total; };

RsStaticOffsets rs_static_offsets(const bte_rs_grid* g) {
    RsStaticOffsets o{};
    o.pitch = (g->n_phiy + 7) / 8 * 8;
    const size_t K = (size_t)g->n_phix, p = (size_t)o.pitch;
    size_t off = 0;
    o.f = off;       off = rs_align(off + 2 * K * p * sizeof(double));
    o.cprime = off;  off = rs_align(off + K * p * sizeof(double));
    o.zvec = off;    off = rs_align(off + K * p * sizeof(double));
    o.ex = off;      off = rs_align(off + K * sizeof(double));
    o.sinx = off;    off = rs_align(off + K * sizeof(double));
    o.gm = off;      off = rs_align(off + p * sizeof(double));
    o.phi = off;     off = rs_align(off + p * sizeof(double));
    o.partial = off; off = rs_align(off + (p / RS_PCR_MT + 1) * 2 * sizeof(double));
    o.obs = off;     off = rs_align(off + sizeof(RsObs));
    o.total = off;
    return o;
}

// In host code `rs_static_scratch` is a host-side stand-in, not a device address: the address a kernel can use comes
// from cudaGetSymbolAddress, asked once per device with that device current.
constexpr int RS_STATIC_MAX_DEVICES = 64;
std::mutex g_rs_static_mutex;
unsigned char* g_rs_static_base[RS_STATIC_MAX_DEVICES] = {};

int rs_static_base(unsigned char** out) {
    int dev = -1;
    RS_CUDA_TRY(cudaGetDevice(&dev));
    if (dev < 0 || dev >= RS_STATIC_MAX_DEVICES) return rs_fail(BTE_EINVAL, "bte_rs_evolve_static: device ordinal out of range");
    std::lock_guard<std::mutex> lock(g_rs_static_mutex);
    if (!g_rs_static_base[dev]) {
        void* ptr = nullptr;
        RS_CUDA_TRY(cudaGetSymbolAddress(&ptr, rs_static_scratch));
        if (!ptr) return rs_fail(BTE_ECUDA, "bte_rs_evolve_static: cudaGetSymbolAddress returned NULL");
        g_rs_static_base[dev] = (unsigned char*)ptr;
    }
    *out = g_rs_static_base[dev];
    return BTE_OK;
}

// the tables of bte_rs_create (eq. 13 split into its phi_x and phi_y parts; C8, C19), formed on the device: no host staging
__global__ void rs_static_tables_kernel(double* ex, double* sinx, double* gm, double* phi, int K, int M1, int pitch,
                                        double pref, double mu, double dx, double centre, double dphi) {
    const int t = blockIdx.x * blockDim.x + threadIdx.x;
    const double PI = 3.14159265358979323846;
    if (t < K) {
        const double x = -PI + dx * t;
        ex[t] = pref * exp(mu * (cos(x) - 1.0));
        sinx[t] = sin(x);
    }
    if (t < pitch) {
        double ph = 0.0, g = 0.0;
        if (t < M1) {
            ph = centre + (t - (M1 - 1) / 2.0) * dphi;
            g = exp(-mu * ph * ph / 2.0);
            if (g < 1e-300) g = 0.0;
        }
        phi[t] = ph;
        gm[t] = g;
    }
}

}  // namespace

extern "C" int bte_rs_evolve_static(const bte_rs_grid* grid, const bte_params* p, const double* f_in, int64_t step0,
                                    int64_t n_steps, double* f_out, bte_obs* obs, void* cuda_stream) {
    if (!grid || !p || !f_out) return rs_fail(BTE_EINVAL, "bte_rs_evolve_static: NULL argument");
    if (!rs_grid_ok(grid)) return rs_fail(BTE_EINVAL, "bte_rs_evolve_static: need 4 <= n_phix <= 4096, n_phiy >= 3, dt > 0");
    if (step0 < 0 || n_steps < 0) return rs_fail(BTE_EINVAL, "bte_rs_evolve_static: step0 < 0 or n_steps < 0");
    if (!f_in && step0 != 0) return rs_fail(BTE_EINVAL, "bte_rs_evolve_static: f_in NULL (start from equilibrium) needs step0 = 0");
    const bool finite = std::isfinite(p->E_dc) && std::isfinite(p->E_omega) && std::isfinite(p->omega) &&
                        std::isfinite(p->B) && std::isfinite(p->mu) && std::isfinite(p->alpha) &&
                        std::isfinite(p->phiy_min) && std::isfinite(p->phiy_max) && std::isfinite(p->kappa_scale);
    if (!finite || !(p->mu > 0.0) || !(p->alpha > 0.0) || !(p->phiy_max > p->phiy_min) || p->n_steps_total < 0 ||
        p->avg_start_step < 0)
        return rs_fail(BTE_EINVAL, "bte_rs_evolve_static: need finite parameters, mu > 0, alpha > 0, phiy_max > phiy_min");
    const RsStaticOffsets off = rs_static_offsets(grid);
    const int K = grid->n_phix, M1 = grid->n_phiy, M = M1 - 1;
    if ((size_t)K * (size_t)off.pitch > RS_STATIC_MAX_POINTS || off.total > RS_STATIC_BYTES) {
        char buf[256];
        snprintf(buf, sizeof buf,
                 "bte_rs_evolve_static: n_phix * pitch = %zu points exceeds the static scratch limit of %zu "
                 "(pitch = n_phiy rounded up to a multiple of 8); use bte_rs_create with a caller-owned workspace",
                 (size_t)K * (size_t)off.pitch, RS_STATIC_MAX_POINTS);
        return rs_fail(BTE_ENOMEM, buf);
    }
    const double dphi = (p->phiy_max - p->phiy_min) / M;
    if (std::fabs(p->B) * grid->dt / dphi >= 2.0)
        return rs_fail(BTE_EUNSTABLE, "bte_rs_evolve_static: |B| dt / dphi >= 2 (scheme unstable, DESIGN.md C11)");
    unsigned char* base = nullptr;
    if (const int rc = rs_static_base(&base)) return rc;
    cudaStream_t stream = (cudaStream_t)cuda_stream;
    const double PI = 3.14159265358979323846;
    const double dx = 2.0 * PI / K;
    bte_rs_ctx c{};                                   // on the stack: what rs_launch reads
    c.grid = *grid; c.params = *p; c.off.pitch = off.pitch; c.ws = (char*)base; c.stream = stream; c.k = step0;
    c.pcr = rs_pcr_kernel_for(K);
    if (c.pcr) RS_CUDA_TRY(cudaFuncSetAttribute(c.pcr, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)rs_pcr_smem(K)));
    RsLayout& L = c.L;
    L.K = K; L.M1 = M1; L.pitch = off.pitch; L.dt = grid->dt; L.dx = dx; L.dphi = dphi;
    L.E_dc = p->E_dc; L.E_omega = p->E_omega; L.omega = p->omega; L.B = p->B; L.kappa_scale = p->kappa_scale;
    L.norm_scale = std::sqrt(p->alpha) * dx * dphi;
    L.f = (double*)(base + off.f); L.cprime = (double*)(base + off.cprime); L.zvec = (double*)(base + off.zvec);
    double* ex = (double*)(base + off.ex);   double* sinx = (double*)(base + off.sinx);
    double* gm = (double*)(base + off.gm);   double* phi = (double*)(base + off.phi);
    L.ex = ex; L.sinx = sinx; L.gm = gm; L.phi = phi;
    L.partial = (double*)(base + off.partial); L.obs = (RsObs*)(base + off.obs);
    // what must start at zero: the running sums and the block counter of the last-block fold
    RS_CUDA_TRY(cudaMemsetAsync(L.obs, 0, sizeof(RsObs), stream));
    const double pref = (1.0 / (2.0 * PI)) * std::sqrt(p->mu / (2.0 * PI * p->alpha)) / bessel_i0_scaled(p->mu);
    const int tn = K > off.pitch ? K : off.pitch;
    rs_static_tables_kernel<<<(unsigned)((tn + 127) / 128), 128, 0, stream>>>(ex, sinx, gm, phi, K, M1, off.pitch, pref, p->mu, dx,
                                                                             0.5 * (p->phiy_min + p->phiy_max), dphi);
    const size_t row = (size_t)M1 * sizeof(double), prow = (size_t)off.pitch * sizeof(double);
    if (f_in) {      // dense [2][K][M1] -> pitched state; the pad columns keep stale values, which no kernel lets through
        RS_CUDA_TRY(cudaMemcpy2DAsync(L.f, prow, f_in, row, row, (size_t)2 * K, cudaMemcpyDeviceToDevice, stream));
    } else {
        const dim3 g((unsigned)((off.pitch + 127) / 128), (unsigned)K);
        rs_init_kernel<<<g, 128, 0, stream>>>(L);
        rs_launch(&c, 2, 0, 0);                       // start-up z^{1/2}, L202
    }
    for (int64_t s = 0; s < n_steps; ++s) {
        if (p->n_steps_total > 0 && c.k >= p->n_steps_total) break;   // frozen
        const int do_avg = (c.k + 1 > p->avg_start_step) ? 1 : 0;
        rs_launch(&c, 0, (long long)c.k, do_avg);     // eq. (40)
        rs_launch(&c, 1, (long long)c.k, 0);          // eq. (41), C5
        c.k += 1;
    }
    RS_CUDA_TRY(cudaGetLastError());
    RS_CUDA_TRY(cudaMemcpy2DAsync(f_out, row, L.f, prow, row, (size_t)2 * K, cudaMemcpyDeviceToDevice, stream));
    if (obs) {
        RsObs o;
        RS_CUDA_TRY(cudaMemcpyAsync(&o, L.obs, sizeof o, cudaMemcpyDeviceToHost, stream));
        RS_CUDA_TRY(cudaStreamSynchronize(stream));
        obs->step = c.k; obs->t = (double)c.k * grid->dt; obs->norm = o.norm; obs->v_dr = o.v_dr;
        obs->sum_v_dt = o.sum_v; obs->sum_vcos_dt = o.sum_c; obs->sum_vsin_dt = o.sum_s; obs->window = o.window;
        obs->edge_leak = 0.0;
    }
    return BTE_OK;
}
