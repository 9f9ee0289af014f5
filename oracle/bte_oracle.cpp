/*
 * bte_oracle.cpp -- TEST INFRASTRUCTURE, NOT THE PRODUCT.
 *
 * Plain, slow, obviously-correct CPU statement (fp64, straight loops) of the Crank-Nicolson + leap-frog
 * time step of arxiv 1401.6047.  It is the oracle the CUDA path is compared with.
 * Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may build,
 * load or call it.  It shares no code, header, table or constant generator with the CUDA library under
 * paper_1401_6047_b200/csrc and neither includes the other.
 *
 * The method is a time iteration, so the oracle is the algorithm step by step, in the paper's order
 * and notation.  Each function cites the passage it follows; the readings taken where the paper is
 * garbled or silent carry the tags (C1..C15) of DESIGN.md "Readings of the paper".
 *
 * Pins (tests/test_oracle_pins.py, run with -m "not gpu"): closed form at B=0 for every (n,m,k), the
 * Esaki-Tsu-type steady drift velocity, norm conservation, relaxation to f0, the B=0 mirror symmetry,
 * the field-reversal mirror, E=0 stationarity of f0 with order-2 convergence, order-2 convergence in
 * dt, the Tucker ac averages, a dense brute-force restatement on tiny grids, checkerboard independence
 * and affinity; the reconstruction of f (eq. 8) against eq. (13) at t = 0 and against a numpy contraction; the
 * pendulum averages (eq. 44-46) against the T = 0 Esaki-Tsu and Tucker closed forms and the energy invariant; the steady
 * drift velocity in CROSSED dc fields at finite temperature against the exact solution of eq. (5) by characteristics
 * (P12: Chambers path integral over the flow (44)-(45) with the Boltzmann f0 of eq. 13; fields of configs 1 and 4).
 * The time-dependent (ac) absolute values of configs 1-4 have no closed form and the paper prints none: for those
 * "parity unpinned" beyond P12 at their dc fields, P9 at B = 0 and the invariants listed above.
 *
 * Build: g++ -std=c++17 -O2 -ffp-contract=off -fopenmp -shared -fPIC (see oracle/build.py).
 * -ffp-contract=off: no FMA contraction, every operation rounds once, in the order written.
 */
#include <cmath>
#include <cstdint>
#include <cstdlib>
#include <cstring>
#include <vector>
#ifdef _OPENMP
#include <omp.h>
#endif

namespace {

const double PI = 3.14159265358979323846;

struct Sim {
    int N, M1;              /* rows n = 0..N (eq. 22), columns m = 0..M, M1 = M+1                       */
    double dt;
    double E_dc, E_omega, omega, B, mu, alpha, phiy_min, phiy_max, kappa_scale;
    int64_t n_steps_total, avg_start_step;
    double dphi;
    std::vector<double> phi;            /* phi_y(m)                                                     */
    std::vector<double> a0;             /* a_n^(0)(m), eq. (15)                                          */
    std::vector<double> ha, hb, fa, fb; /* whole grid z_h and fractional grid z_f, eq. (39)-(41)         */
    std::vector<double> sa, sb;         /* snapshot used only by the start-up step                       */
    std::vector<float> cf, gf;          /* precision 2: c_n and g_m = exp(-mu phi^2/2) rounded to fp32   */
    int64_t step;
    double norm, v_dr, sum_v, sum_c, sum_s, window;
    /* steady-state detection and averaging policy (C23); steady_tol = 0: off */
    double steady_tol;
    int n_avg_periods, min_relax_periods;
    int64_t period_steps, window_steps, interval_pos, intervals_done, window_left, steady_step;
    double interval_sum, previous_mean;
    int phase;              /* 0 relaxing, 1 averaging, 2 finished */
    int threads;
    int precision;          /* 0: fp64 (default); 1: state stored as fp32, arithmetic fp64; 2: fp32 throughout (NEXT-4) */
};

inline size_t idx(const Sim* s, int n, int m) { return (size_t)n * (size_t)s->M1 + (size_t)m; }

/* Boundary conditions (22)-(23): a = 0 outside n in [0..N], m in [0..M]; b = 0 outside n in [1..N],
 * m in [0..M] (reading C3: b_0 == 0 because sin(0*phi_x) = 0).                                          */
inline double rd_a(const Sim* s, const double* a, int n, int m) {
    if (n < 0 || n > s->N || m < 0 || m >= s->M1) return 0.0;
    return a[idx(s, n, m)];
}
inline double rd_b(const Sim* s, const double* b, int n, int m) {
    if (n < 1 || n > s->N || m < 0 || m >= s->M1) return 0.0;
    return b[idx(s, n, m)];
}

/* E(t) = E_dc + E_omega cos(omega t). */
inline double field_E(const Sim* s, double t) { return s->E_dc + s->E_omega * std::cos(s->omega * t); }

/*
 * Operator T of eq. (38): advance grid X in place by `delta`, the derivative terms A, B of eq. (30)-(31)
 * taken from grid S, the rotation term at time ta (explicit half) and tb (implicit half).
 *   kappa   = kappa_scale * B * delta / (4 dphi)                eq. (30)-(31) prefactor, reading C4
 *   nu, xi  = 1 +- delta/2                                      eq. (34)-(35)
 *   mu^t    = n * beta^t_m * delta / 2, beta = E + B phi_y(m)   eq. (28)-(29)
 *   g, h                                                       eq. (36)-(37)
 *   a', b'                                                     eq. (32) and (33) with the sign of (33)
 *                                                              corrected (reading C2: Cramer's rule on
 *                                                              (24)+(26), (25)+(27))
 * X and S must not alias (the start-up step passes a snapshot).
 */
void apply_T(const Sim* s, double delta, double* Xa, double* Xb, const double* Sa, const double* Sb,
             double ta, double tb) {
    const int N = s->N, M1 = s->M1;
    const double kappa = s->kappa_scale * s->B * delta / (4.0 * s->dphi);
    const double nu = 1.0 + delta / 2.0;
    const double xi = 1.0 - delta / 2.0;
    const double Ea = field_E(s, ta);
    const double Eb = field_E(s, tb);
#pragma omp parallel for schedule(static) num_threads(s->threads)
    for (int n = 0; n <= N; ++n) {
        for (int m = 0; m < M1; ++m) {
            const double beta_a = Ea + s->B * s->phi[m];
            const double beta_b = Eb + s->B * s->phi[m];
            const double mu_a = n * beta_a * delta / 2.0;
            const double mu_b = n * beta_b * delta / 2.0;
            const double chi = (n == 1) ? 2.0 : 1.0; /* eq. (11) */
            const double Bt = kappa * (rd_b(s, Sb, n + 1, m + 1) - rd_b(s, Sb, n + 1, m - 1) -
                                       rd_b(s, Sb, n - 1, m + 1) + rd_b(s, Sb, n - 1, m - 1));
            const double At = kappa * (chi * (rd_a(s, Sa, n - 1, m + 1) - rd_a(s, Sa, n - 1, m - 1)) -
                                       rd_a(s, Sa, n + 1, m + 1) + rd_a(s, Sa, n + 1, m - 1));
            const size_t i = idx(s, n, m);
            const double a = Xa[i];
            const double b = Xb[i];
            const double g = a * xi - b * mu_a + Bt + s->a0[i] * delta;
            const double h = b * xi + a * mu_a + At;
            const double det = nu * nu + mu_b * mu_b;
            Xa[i] = (g * nu - h * mu_b) / det;
            Xb[i] = (n >= 1) ? (g * mu_b + h * nu) / det : 0.0;
            if (s->precision == 1) { /* the state lives in fp32 storage: every new value is rounded once */
                Xa[i] = (double)(float)Xa[i];
                Xb[i] = (double)(float)Xb[i];
            }
        }
    }
}

/* The same operator T with every quantity and every operation in fp32, "all code used float data type"
 * (PAPER.md:L311), SURVEY 8(f) NEXT-4.  The arrays hold values that are exactly representable in fp32.  Scalars that
 * do not depend on the lattice point (E(t), kappa, nu, xi) are formed in fp64 and rounded once; c_n and the Gaussian
 * factor g_m are rounded to fp32 and a^(0) delta is formed as c_n (g_m delta).  Operation order as written, one
 * rounding per operation (-ffp-contract=off), IEEE division.                                                      */
void apply_T_f32(const Sim* s, double delta_d, double* Xa, double* Xb, const double* Sa, const double* Sb, double ta,
                 double tb, const std::vector<float>& cf, const std::vector<float>& gf) {
    const int N = s->N, M1 = s->M1;
    const float delta = (float)delta_d;
    const float kappa = (float)(s->kappa_scale * s->B * delta_d / (4.0 * s->dphi));
    const float nu = (float)(1.0 + delta_d / 2.0);
    const float xi = (float)(1.0 - delta_d / 2.0);
    const float Ea = (float)field_E(s, ta);
    const float Eb = (float)field_E(s, tb);
    const float Bf = (float)s->B;
#pragma omp parallel for schedule(static) num_threads(s->threads)
    for (int n = 0; n <= N; ++n) {
        const float nf = (float)n;
        for (int m = 0; m < M1; ++m) {
            const float ph = (float)s->phi[m];
            const float beta_a = Ea + Bf * ph;
            const float beta_b = Eb + Bf * ph;
            const float mu_a = nf * beta_a * delta / 2.0f;
            const float mu_b = nf * beta_b * delta / 2.0f;
            const float chi = (n == 1) ? 2.0f : 1.0f;
            const float Bt = kappa * ((float)rd_b(s, Sb, n + 1, m + 1) - (float)rd_b(s, Sb, n + 1, m - 1) -
                                      (float)rd_b(s, Sb, n - 1, m + 1) + (float)rd_b(s, Sb, n - 1, m - 1));
            const float At = kappa * (chi * ((float)rd_a(s, Sa, n - 1, m + 1) - (float)rd_a(s, Sa, n - 1, m - 1)) -
                                      (float)rd_a(s, Sa, n + 1, m + 1) + (float)rd_a(s, Sa, n + 1, m - 1));
            const size_t i = idx(s, n, m);
            const float a = (float)Xa[i];
            const float b = (float)Xb[i];
            const float src = cf[n] * (gf[m] * delta);
            const float g = a * xi - b * mu_a + Bt + src;
            const float h = b * xi + a * mu_a + At;
            const float det = nu * nu + mu_b * mu_b;
            Xa[i] = (double)((g * nu - h * mu_b) / det);
            Xb[i] = (n >= 1) ? (double)((g * mu_b + h * nu) / det) : 0.0;
        }
    }
}

void run_T(const Sim* s, double delta, double* Xa, double* Xb, const double* Sa, const double* Sb, double ta,
           double tb) {
    if (s->precision == 2) apply_T_f32(s, delta, Xa, Xb, Sa, Sb, ta, tb, s->cf, s->gf);
    else apply_T(s, delta, Xa, Xb, Sa, Sb, ta, tb);
}

/* phi_y lattice (reading C8) and equilibrium coefficients, eq. (15)-(16) with sigma(0) = 1/2,
 * sigma(n>=1) = 1 (reading C1).  I_n(mu)/I_0(mu) from the C++17 library routine (reading C13).
 * Values of the Gaussian factor below 1e-300 are set to 0 (input-recipe clamp, C19).        */
void fill_equilibrium(Sim* s) {
    const int N = s->N, M1 = s->M1, M = M1 - 1;
    s->dphi = (s->phiy_max - s->phiy_min) / M;
    s->phi.resize(M1);
    for (int m = 0; m < M1; ++m)
        s->phi[m] = 0.5 * (s->phiy_min + s->phiy_max) + (m - M / 2.0) * s->dphi;
    const double i0 = std::cyl_bessel_i(0.0, s->mu);
    const double pref = std::sqrt(s->mu / (2.0 * PI * s->alpha));
    s->a0.assign((size_t)(N + 1) * M1, 0.0);
    s->cf.assign(N + 1, 0.0f);
    s->gf.assign(M1, 0.0f);
    for (int n = 0; n <= N; ++n) {
        const double r = std::cyl_bessel_i((double)n, s->mu) / i0;
        const double c = (n == 0) ? (1.0 / (2.0 * PI)) * pref : (r / PI) * pref;
        for (int m = 0; m < M1; ++m) {
            double gm = std::exp(-s->mu * s->phi[m] * s->phi[m] / 2.0);
            if (gm < 1e-300) gm = 0.0;
            s->a0[idx(s, n, m)] = c * gm;
            s->gf[m] = (float)gm;
        }
        s->cf[n] = (float)c;
    }
}

/* Observables on the whole grid: eq. (12) and eq. (20) by the rectangle rule (reading C10). */
void reduce_observables(Sim* s) {
    double sa = 0.0, sb = 0.0;
    for (int m = 0; m < s->M1; ++m) sa += s->ha[idx(s, 0, m)];
    if (s->N >= 1)
        for (int m = 0; m < s->M1; ++m) sb += s->hb[idx(s, 1, m)];
    s->norm = 2.0 * PI * std::sqrt(s->alpha) * s->dphi * sa;
    s->v_dr = PI * std::sqrt(s->alpha) * s->dphi * sb;
}

} // namespace

extern "C" {

struct oracle_params {
    double E_dc, E_omega, omega, B, mu, alpha, phiy_min, phiy_max, kappa_scale;
    int64_t n_steps_total, avg_start_step;
};

struct oracle_obs {
    int64_t step;
    double t, norm, v_dr, sum_v_dt, sum_vcos_dt, sum_vsin_dt, window, edge_leak;
};

void* oracle_create(int32_t n_harm, int32_t n_phiy, double dt, const oracle_params* p, int32_t threads) {
    if (n_harm < 1 || n_phiy < 3 || !(dt > 0) || !(p->mu > 0) || !(p->alpha > 0) ||
        !(p->phiy_max > p->phiy_min))
        return nullptr;
    Sim* s = new Sim();
    s->N = n_harm; s->M1 = n_phiy; s->dt = dt;
    s->E_dc = p->E_dc; s->E_omega = p->E_omega; s->omega = p->omega; s->B = p->B; s->mu = p->mu;
    s->alpha = p->alpha; s->phiy_min = p->phiy_min; s->phiy_max = p->phiy_max;
    s->kappa_scale = p->kappa_scale;
    s->n_steps_total = p->n_steps_total; s->avg_start_step = p->avg_start_step;
    s->threads = threads > 0 ? threads : 1;
    s->precision = 0;
    s->steady_tol = 0.0; s->n_avg_periods = 0; s->min_relax_periods = 0; s->period_steps = 0; s->window_steps = 0;
    s->interval_pos = s->intervals_done = s->window_left = s->steady_step = 0;
    s->interval_sum = s->previous_mean = 0.0; s->phase = 0;
    fill_equilibrium(s);
    const size_t P = (size_t)(s->N + 1) * s->M1;
    s->ha.assign(P, 0.0); s->hb.assign(P, 0.0); s->fa.assign(P, 0.0); s->fb.assign(P, 0.0);
    s->step = 0; s->norm = s->v_dr = s->sum_v = s->sum_c = s->sum_s = s->window = 0.0;
    return s;
}

void oracle_destroy(void* h) { delete (Sim*)h; }

/* NEXT-4: 0 = fp64 (default), 1 = state stored in fp32 / arithmetic fp64, 2 = fp32 throughout.  Call before
 * oracle_init_equilibrium.                                                                                    */
void oracle_set_precision(void* h, int32_t precision) { ((Sim*)h)->precision = precision; }

/* Initial condition a = a^(0), b = 0 and start-up of the fractional grid: z^{1/2} by
 * (38) with time step dt/2 (reading C6: delta = dt/2 everywhere, stencil from z^0,
 * field times 0 and dt/2).                                                                             */
void oracle_init_equilibrium(void* h) {
    Sim* s = (Sim*)h;
    s->ha = s->a0;
    if (s->precision == 1)
        for (double& x : s->ha) x = (double)(float)x;
    if (s->precision == 2)
        for (int n = 0; n <= s->N; ++n)
            for (int m = 0; m < s->M1; ++m) s->ha[idx(s, n, m)] = (double)(s->cf[n] * s->gf[m]);
    std::fill(s->hb.begin(), s->hb.end(), 0.0);
    s->fa = s->ha; s->fb = s->hb;
    run_T(s, s->dt / 2.0, s->fa.data(), s->fb.data(), s->ha.data(), s->hb.data(), 0.0, s->dt / 2.0);
    s->step = 0; s->sum_v = s->sum_c = s->sum_s = s->window = 0.0;
    reduce_observables(s);
}

/* Recompute the fractional grid from the current whole grid exactly as the start-up does, treating the
 * current whole-grid state as z^0 at t = 0 (test helper for arbitrary initial states).                 */
void oracle_startup_from_whole(void* h) {
    Sim* s = (Sim*)h;
    s->fa = s->ha; s->fb = s->hb;
    run_T(s, s->dt / 2.0, s->fa.data(), s->fb.data(), s->ha.data(), s->hb.data(), 0.0, s->dt / 2.0);
    s->step = 0; s->sum_v = s->sum_c = s->sum_s = s->window = 0.0;
    reduce_observables(s);
}

/* n_steps leap-frog steps, eq. (40)-(41): whole grid with the stencil of the fractional grid, then the
 * fractional grid with the stencil of the NEW whole grid (reading C5).  Times are formed by
 * multiplication, never accumulated (reading C14).  After each step the observables (12), (20) and,
 * for steps k+1 > avg_start_step, the running sums of eq. (17) (reading C9).  v_trace / norm_trace are
 * optional per-step outputs (length n_steps).                                                          */
void oracle_step(void* h, int64_t n_steps, double* v_trace, double* norm_trace) {
    Sim* s = (Sim*)h;
    for (int64_t j = 0; j < n_steps; ++j) {
        if (s->n_steps_total > 0 && s->step >= s->n_steps_total) {
            if (v_trace) v_trace[j] = s->v_dr;
            if (norm_trace) norm_trace[j] = s->norm;
            continue;
        }
        const double k = (double)s->step;
        run_T(s, s->dt, s->ha.data(), s->hb.data(), s->fa.data(), s->fb.data(), k * s->dt,
                (k + 1.0) * s->dt);
        run_T(s, s->dt, s->fa.data(), s->fb.data(), s->ha.data(), s->hb.data(), (k + 0.5) * s->dt,
                (k + 1.5) * s->dt);
        s->step += 1;
        const double t = (double)s->step * s->dt;
        reduce_observables(s);
        bool accumulate = s->step > s->avg_start_step;          /* fixed window, reading C9 */
        if (s->steady_tol > 0.0) {
            /* Reading C23 of PAPER.md:L103 ("let the system relax ... then compute averages over the period"): the mean
             * drift velocity of every interval of P steps (one ac period) is compared with that of the interval
             * before; once two consecutive means agree to steady_tol (not before max(2, min_relax) intervals) the sums
             * of eq. (17) run over the next round(n_avg_periods * period / dt) steps, then stop for good. */
            accumulate = false;
            if (s->phase == 1) {
                accumulate = true;
                s->window_left -= 1;
                if (s->window_left == 0) s->phase = 2;
            } else if (s->phase == 0) {
                s->interval_sum += s->v_dr;
                s->interval_pos += 1;
                if (s->interval_pos == s->period_steps) {
                    const double mean = s->interval_sum / (double)s->period_steps;
                    s->intervals_done += 1;
                    const double scale = std::max(std::max(std::fabs(mean), std::fabs(s->previous_mean)), 1e-3);
                    const int64_t need = std::max(2, s->min_relax_periods);
                    if (s->intervals_done >= need && std::fabs(mean - s->previous_mean) <= s->steady_tol * scale) {
                        s->phase = 1;
                        s->window_left = s->window_steps;
                        s->steady_step = s->step;
                    }
                    s->previous_mean = mean;
                    s->interval_sum = 0.0;
                    s->interval_pos = 0;
                }
            }
        }
        if (accumulate) {
            s->sum_v += s->v_dr * s->dt;
            s->sum_c += s->v_dr * std::cos(s->omega * t) * s->dt;
            s->sum_s += s->v_dr * std::sin(s->omega * t) * s->dt;
            s->window += s->dt;
        }
        if (v_trace) v_trace[j] = s->v_dr;
        if (norm_trace) norm_trace[j] = s->norm;
    }
}

/* Switch the steady-state policy on (tol > 0) or off; resets its bookkeeping.  P = one ac period in steps, or one
 * relaxation time for a dc system.  (A finished system keeps evolving when stepped; only its sums are final.) */
void oracle_set_steady_policy(void* h, double tol, int32_t n_avg_periods, int32_t min_relax_periods) {
    Sim* s = (Sim*)h;
    const double pi = 3.14159265358979323846;
    const double w = std::fabs(s->omega);
    const double P = w > 0.0 ? 2.0 * pi / (w * s->dt) : 1.0 / s->dt;
    s->period_steps = std::max<int64_t>(1, std::llround(P));
    s->window_steps = std::max<int64_t>(1, std::llround((double)n_avg_periods * P));   /* rounded once, not per period */
    s->steady_tol = tol; s->n_avg_periods = n_avg_periods; s->min_relax_periods = min_relax_periods;
    s->interval_pos = 0; s->intervals_done = 0; s->window_left = 0; s->steady_step = 0;
    s->interval_sum = 0.0; s->previous_mean = 0.0; s->phase = 0;
}

void oracle_steady_info(void* h, int64_t* steady_step, int32_t* phase) {
    Sim* s = (Sim*)h;
    *steady_step = s->steady_step;
    *phase = s->phase;
}

void oracle_observables(void* h, oracle_obs* o) {
    Sim* s = (Sim*)h;
    o->step = s->step;
    o->t = (double)s->step * s->dt;
    o->norm = s->norm; o->v_dr = s->v_dr;
    o->sum_v_dt = s->sum_v; o->sum_vcos_dt = s->sum_c; o->sum_vsin_dt = s->sum_s; o->window = s->window;
    o->edge_leak = (s->N >= 1) ? std::fabs(s->hb[idx(s, 1, 0)]) + std::fabs(s->hb[idx(s, 1, s->M1 - 1)])
                               : 0.0;
}

/* grid: 0 = whole, 1 = fractional.  a, b: (N+1) x (M+1) row-major, m fastest. */
void oracle_get_state(void* h, int32_t grid, double* a, double* b) {
    Sim* s = (Sim*)h;
    const size_t bytes = sizeof(double) * (size_t)(s->N + 1) * s->M1;
    std::memcpy(a, grid == 0 ? s->ha.data() : s->fa.data(), bytes);
    std::memcpy(b, grid == 0 ? s->hb.data() : s->fb.data(), bytes);
}

void oracle_set_state(void* h, int32_t grid, const double* a, const double* b) {
    Sim* s = (Sim*)h;
    const size_t bytes = sizeof(double) * (size_t)(s->N + 1) * s->M1;
    std::memcpy(grid == 0 ? s->ha.data() : s->fa.data(), a, bytes);
    std::memcpy(grid == 0 ? s->hb.data() : s->fb.data(), b, bytes);
    if (grid == 0) reduce_observables(s);
}

void oracle_get_equilibrium(void* h, double* phi, double* a0) {
    Sim* s = (Sim*)h;
    std::memcpy(phi, s->phi.data(), sizeof(double) * s->M1);
    std::memcpy(a0, s->a0.data(), sizeof(double) * (size_t)(s->N + 1) * s->M1);
}

/* One bare application of T (eq. 38) to grid `target` (0 whole, 1 fractional) with the stencil taken
 * from the OTHER grid, time step delta, field times ta, tb.  Test hook for the brute-force,
 * checkerboard and affinity pins.                                                                      */
void oracle_apply_T(void* h, int32_t target, double delta, double ta, double tb) {
    Sim* s = (Sim*)h;
    if (target == 0)
        run_T(s, delta, s->ha.data(), s->hb.data(), s->fa.data(), s->fb.data(), ta, tb);
    else
        run_T(s, delta, s->fa.data(), s->fb.data(), s->ha.data(), s->hb.data(), ta, tb);
}

/* The distribution function itself, eq. (8): f(phi_x, phi_y) = sum_n a_n cos(n phi_x) + b_n sin(n phi_x), written
 * out as that sum (n ascending) on K equidistant phi_x = -pi + 2 pi i / K, i = 0..K-1, for every phi_y lattice
 * point.  grid: 0 = whole, 1 = fractional.  f: K x (M+1) row-major, m fastest.  (pinned by
 * eq. (13) at t = 0 in tests/test_oracle_pins.py.)                                                          */
void oracle_reconstruct_pdf(void* h, int32_t grid, int32_t K, double* f) {
    Sim* s = (Sim*)h;
    const double PI = 3.14159265358979323846;
    const double* a = grid == 0 ? s->ha.data() : s->fa.data();
    const double* b = grid == 0 ? s->hb.data() : s->fb.data();
    for (int i = 0; i < K; ++i) {
        const double x = -PI + 2.0 * PI * i / K;
        for (int m = 0; m < s->M1; ++m) {
            double acc = 0.0;
            for (int n = 0; n <= s->N; ++n)
                acc += a[idx(s, n, m)] * std::cos(n * x) + b[idx(s, n, m)] * std::sin(n * x);
            f[(size_t)i * s->M1 + m] = acc;
        }
    }
}

/* ---- the zero-temperature limit, eq. (44)-(46) ---------------------
 * A single electron starts at (phi_x, phi_y) = (0, 0) (f0 -> delta function, L217) at time t0 and follows
 *     d phi_x / dt = E(t) + B phi_y            (44)        E(t) = E_dc + E_omega cos(omega t)   (L99)
 *     d phi_y / dt = -B sin(phi_x)             (45)
 * Its velocity along x is sin(phi_x) (dispersion (3) in the units of (4)).  Dissipation re-enters through the
 * exponential memory (46): v_dr(t) = int_{-inf}^{t} sin phi_x(t; t0) e^{-(t - t0)} dt0.  Averaged over one ac period
 * (t0 -> start phase, s = t - t0):
 *     <v_dr>          = (1/T) int_0^T dt0 int_0^inf ds e^{-s} sin phi_x(t0 + s; t0)
 *     <v_dr cos wt>   = (1/T) int_0^T dt0 int_0^inf ds e^{-s} sin phi_x(t0 + s; t0) cos(w (t0 + s))     (17), I1/I0 -> 1
 * The paper gives no discretisation ("can be trivially solved numerically", L235); reading taken (C20):
 * classical RK4 with step h for (44)-(45), composite Simpson on the RK4 nodes s_k = k h, k = 0..n_rk (n_rk even,
 * memory cut at n_rk h), rectangle rule over n_phase equidistant start phases t0_j = j T / n_phase (periodic
 * integrand).  Without an ac field (E_omega = 0 or omega = 0) one start phase, t0 = 0.
 * out[0..2] = <v_dr>, <v_dr cos wt>, <v_dr sin wt>.                                                             */
static void pendulum_rhs(double Edc, double Ew, double w, double B, double t, double px, double py, double* dx,
                         double* dy) {
    *dx = (Edc + Ew * std::cos(w * t)) + B * py;
    *dy = -B * std::sin(px);
}

void oracle_pendulum_averages(double Edc, double Ew, double w, double B, int32_t n_phase, double h, int32_t n_rk,
                              double* out) {
    const double PI = 3.14159265358979323846;
    const bool ac = (Ew != 0.0) && (w != 0.0);
    const int P = ac ? n_phase : 1;
    const double T = ac ? 2.0 * PI / w : 0.0;
    double sum0 = 0.0, sumc = 0.0, sums = 0.0;
    for (int j = 0; j < P; ++j) {
        const double t0 = ac ? T * j / P : 0.0;
        double px = 0.0, py = 0.0, I0 = 0.0, Ic = 0.0, Is = 0.0;
        for (int k = 0; k <= n_rk; ++k) {
            const double s = k * h, t = t0 + s;
            const double wgt = (k == 0 || k == n_rk) ? 1.0 : ((k & 1) ? 4.0 : 2.0);
            const double g = std::exp(-s) * std::sin(px);
            I0 += wgt * g;
            Ic += wgt * g * std::cos(w * t);
            Is += wgt * g * std::sin(w * t);
            if (k == n_rk) break;
            double k1x, k1y, k2x, k2y, k3x, k3y, k4x, k4y;
            pendulum_rhs(Edc, Ew, w, B, t, px, py, &k1x, &k1y);
            pendulum_rhs(Edc, Ew, w, B, t + 0.5 * h, px + 0.5 * h * k1x, py + 0.5 * h * k1y, &k2x, &k2y);
            pendulum_rhs(Edc, Ew, w, B, t + 0.5 * h, px + 0.5 * h * k2x, py + 0.5 * h * k2y, &k3x, &k3y);
            pendulum_rhs(Edc, Ew, w, B, t + h, px + h * k3x, py + h * k3y, &k4x, &k4y);
            px += (h / 6.0) * (k1x + 2.0 * k2x + 2.0 * k3x + k4x);
            py += (h / 6.0) * (k1y + 2.0 * k2y + 2.0 * k3y + k4y);
        }
        sum0 += I0 * (h / 3.0);
        sumc += Ic * (h / 3.0);
        sums += Is * (h / 3.0);
    }
    out[0] = sum0 / P;
    out[1] = sumc / P;
    out[2] = sums / P;
}

/* Test hook: the trajectory itself, n_rk + 1 nodes from (0, 0) at t0 (for the energy-invariant pin). */
void oracle_pendulum_trajectory(double Edc, double Ew, double w, double B, double t0, double h, int32_t n_rk,
                                double* px_out, double* py_out) {
    double px = 0.0, py = 0.0;
    for (int k = 0; k <= n_rk; ++k) {
        px_out[k] = px;
        py_out[k] = py;
        if (k == n_rk) break;
        const double t = t0 + k * h;
        double k1x, k1y, k2x, k2y, k3x, k3y, k4x, k4y;
        pendulum_rhs(Edc, Ew, w, B, t, px, py, &k1x, &k1y);
        pendulum_rhs(Edc, Ew, w, B, t + 0.5 * h, px + 0.5 * h * k1x, py + 0.5 * h * k1y, &k2x, &k2y);
        pendulum_rhs(Edc, Ew, w, B, t + 0.5 * h, px + 0.5 * h * k2x, py + 0.5 * h * k2y, &k3x, &k3y);
        pendulum_rhs(Edc, Ew, w, B, t + h, px + h * k3x, py + h * k3y, &k4x, &k4y);
        px += (h / 6.0) * (k1x + 2.0 * k2x + 2.0 * k3x + k4x);
        py += (h / 6.0) * (k1y + 2.0 * k2y + 2.0 * k3y + k4y);
    }
}

int32_t oracle_max_threads(void) {
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}

} /* extern "C" */
