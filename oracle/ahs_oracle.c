/*
 * ahs_oracle.c -- TEST INFRASTRUCTURE, NOT PRODUCT CODE.
 *
 * Plain, slow fp64 CPU oracle for the hot path of arXiv 1809.00995
 * (Correia & Martins, "Abelian-Higgs Cosmic String Evolution with CUDA"): the damped
 * staggered-leapfrog update of (phi, Pi, A_i, E_i) and the network diagnostics
 * (plaquette winding, Lagrangian-weighted <v^2>, Gauss-law residual).
 *
 * Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may
 * build, load or call this file.  It shares no code, header, table or helper with the CUDA
 * library under paper_1809_00995_b200/csrc/ and neither includes the other.
 *
 * It follows PAPER.md section 2 (L29-L99) step by step, in the paper's order and notation, with the
 * readings of DESIGN.md "Readings of the paper" (R1..R12) where the text is silent or garbled:
 *   - link phase  U_i^x = exp(-i q theta_i^x), q = +1 pinned (R1);
 *   - theta_i = e0*dx*A_i and eps_i = d theta_i / d eta are the stored "A" and "E" (L44, L62; R5);
 *   - a(tau) = (tau/tau_ref)^m (L224; R3);  e(a) = e0 a^(s-1), lambda(a) = lambda0 a^(2(s-1)) (Eq. 8).
 *
 * Field container ("f10"): 10 contiguous arrays of N^3 doubles, in the order
 *   phi_re, phi_im, Pi_re, Pi_im, theta_0, theta_1, theta_2, eps_0, eps_1, eps_2,
 * site index = x + N*(y + N*z), x fastest; direction 0,1,2 = x,y,z.
 * "Snapshot after n steps" = { phi^n, theta^n at tau_n = tau0 + n*dt ; Pi^(n-1/2), eps^(n-1/2) }.
 *
 * Pins (tests/test_oracle_pins.py, run with -m "not gpu"): every function below is pinned by
 * something other than itself -- see the per-function "pinned by" notes and DESIGN.md.
 *
 * Threads.  The loops over sites are independent per site (the kicks read level-n phi, theta only and write
 * the site's own Pi, eps), so their outer z loop carries an OpenMP "parallel for": the fields are bit-identical
 * for any thread count.  Floating-point sums (diagnostics) are formed per z-plane in x-fastest order and the
 * plane sums are added in z order, whatever the thread count, so every result is independent of it as well
 * (pinned by test_oracle_is_independent_of_the_thread_count).  One thread unless aho_set_threads() says
 * otherwise ("oracle, 1 core" and "oracle, all cores").
 *
 * Build: gcc -O2 -ffp-contract=off -fopenmp -fPIC -shared -o libahs_oracle.so ahs_oracle.c -lm
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

/* number of threads the site loops use (default 1); returns the number actually in effect */
static int aho_threads = 1;
int32_t aho_set_threads(int32_t n)
{
#ifdef _OPENMP
    if (n <= 0) n = omp_get_num_procs();
    aho_threads = n;
#else
    (void)n;
    aho_threads = 1;
#endif
    return aho_threads;
}

typedef struct {
    int32_t N;        /* lattice is N^3, periodic (any N >= 3)                                  */
    int32_t q;        /* +1 pinned convention U = exp(-i theta); -1 = Eqs. 4,5,11 as printed   */
    double dx;        /* lattice spacing Delta x   (L51)                                        */
    double dt;        /* conformal time step Delta eta (L51)                                    */
    double lambda0;   /* lambda_0 (Eq. 8)                                                  */
    double e0;        /* e_0      (Eq. 8)                                                  */
    double sigma;     /* vacuum expectation value (L36, L51)                                    */
    double m;         /* a ~ tau^m : 1 radiation, 2 matter (L224)                               */
    double s;         /* core-width parameter of Eq. 8 (L68-70)                                 */
    double tau0;      /* conformal time of step 0                                               */
    double tau_ref;   /* a(tau) = (tau/tau_ref)^m ; normalisation not given in the paper (R3)   */
    double c_B;       /* factor on the plaquette sum of Eq. 2; 1 = consistent with Eq. 5 (R2)   */
    double c_E;       /* factor on the electric term of Eq. 2 IN THE WEIGHT; 1 = eps = d theta/d eta (R5);
                         (dt/dx)^2 = the rescaling "E -> e dt E" of L44 read literally (R21)          */
    int32_t ns;       /* knots of a time-dependent s(tau) (L66-70: core growth, then s = 1); 0 = constant s     */
    int32_t pad_;
    const double* sched_tau;   /* ns increasing conformal times                                      (R23)      */
    const double* sched_s;     /* s at the knots; linear in between, constant outside                           */
} aho_params;

typedef struct {
    uint64_t n_pierced;       /* number of plaquettes with W != 0 (Eq. 11)              */
    uint64_t sum_abs_w;       /* sum of |W| over all 3 N^3 plaquettes                           */
    double L;                 /* (pi/6) * dx * n_pierced (L93)                                  */
    double xi;                /* sqrt((N dx)^3 / L) ; +inf if n_pierced == 0 (L88)              */
    double v2_num;            /* sum_x |Pi|^2 * Lag   (Eq. 10 numerator, weight = Eq. 2)        */
    double v2_den;            /* sum_x |D phi|^2 * Lag (Eq. 10 denominator)                     */
    double v2;                /* 2R/(1+R), R = num/den (Eq. 9)                                  */
    double mean_lagrangian;   /* sum_x Lag / N^3                                                */
    double gauss_max;         /* max_x |g^x|                                                    */
    double gauss_rhs_rms;     /* rms_x of 2 q dx^2 e0^2 a_h^(2s) Im[conj(phi) Pi]               */
    int32_t nonfinite;        /* 1 if any of the 10 N^3 field values is not finite              */
    int32_t pad_;
    double v2v_num;           /* sum_x |Pi|^2 * Vp    (Eq. 10 with the potential weight, L86)   */
    double v2v_den;           /* sum_x |D phi|^2 * Vp                                           */
    double v2_V;              /* 2R/(1+R), R = v2v_num / v2v_den (Eq. 9)                        */
    double xi_L;              /* sqrt(-mu / mean Lag), mu = 2 pi sigma^2 (Eq. 9; R20); NaN if mean Lag >= 0 */
    double eos_num;           /* sum_x p^x Lag^x    (Eq. 12: Lagrangian-weighted pressure; p, rho per R22)      */
    double eos_den;           /* sum_x rho^x Lag^x                                                              */
    double v2_omega;          /* (1 + 3 eos_num / eos_den) / 2   (Eq. 12)                               */
} aho_diag;

static const double AHO_TWO_PI  = 6.283185307179586476925286766559;
static const double AHO_INV_2PI = 0.15915494309189535; /* R7: ties-to-even of delta * INV_2PI  */

/* ----------------------------------------------------------------------------------------------
 * Philox4x32-10 (Salmon, Moraes, Dror, Shaw 2011), the counter-based generator both paths
 * implement separately.
 * pinned by: the Random123 known-answer vectors in tests/golden/philox4x32_10_kat.txt and an
 * independent implementation (ATen's philox engine header, compiled in the test).
 * -------------------------------------------------------------------------------------------- */
void aho_philox4x32_10(const uint32_t ctr[4], const uint32_t key[2], uint32_t out[4])
{
    const uint32_t M0 = 0xD2511F53u, M1 = 0xCD9E8D57u; /* round multipliers       */
    const uint32_t W0 = 0x9E3779B9u, W1 = 0xBB67AE85u; /* Weyl key increments     */
    uint32_t c0 = ctr[0], c1 = ctr[1], c2 = ctr[2], c3 = ctr[3];
    uint32_t k0 = key[0], k1 = key[1];
    for (int round = 0; round < 10; ++round) {
        uint64_t p0 = (uint64_t)M0 * (uint64_t)c0;
        uint64_t p1 = (uint64_t)M1 * (uint64_t)c2;
        uint32_t hi0 = (uint32_t)(p0 >> 32), lo0 = (uint32_t)p0;
        uint32_t hi1 = (uint32_t)(p1 >> 32), lo1 = (uint32_t)p1;
        uint32_t n0 = hi1 ^ c1 ^ k0;
        uint32_t n1 = lo1;
        uint32_t n2 = hi0 ^ c3 ^ k1;
        uint32_t n3 = lo0;
        c0 = n0; c1 = n1; c2 = n2; c3 = n3;
        k0 += W0; k1 += W1;          /* key is bumped between rounds */
    }
    out[0] = c0; out[1] = c1; out[2] = c2; out[3] = c3;
}

/* u(hi,lo) = (((uint64)hi << 32 | lo) >> 11) * 2^-53, in [0,1) */
static double aho_u53(uint32_t hi, uint32_t lo)
{
    uint64_t w = ((uint64_t)hi << 32) | (uint64_t)lo;
    return (double)(w >> 11) * (1.0 / 9007199254740992.0);
}

/* ----------------------------------------------------------------------------------------------
 * Initial condition: "the scalar field phi is set to have a random phase, its
 * norm is set to unity (given sigma=1) and all other field variables are set to zero".
 *   kind 0: phi = sigma * exp(i 2 pi u(r0,r1)),   (r0..r3) = Philox(counter=(site,0), key=seed)
 *   kind 1: Gaussian (BASELINE config 3; not in the paper): Box-Muller,
 *           u1 = u(r0,r1) + 2^-54, u2 = u(r2,r3), phi = sigma/sqrt2 * sqrt(-2 ln u1) * exp(i 2 pi u2)
 * pinned by: Philox KAT; |phi| = sigma exactly-to-rounding; pierced fraction 1/3 (four i.i.d.
 * uniform corner phases); Gauss residual identically 0 at n = 0; sample moments of kind 1 and two
 * sites of kind 1 by hand (Box-Muller written out in Python from the Philox words).
 * -------------------------------------------------------------------------------------------- */
static void aho_ic_site(const aho_params* p, const uint32_t key[2], int64_t site, int32_t kind, double* re, double* im)
{
    uint32_t ctr[4] = { (uint32_t)((uint64_t)site & 0xffffffffu), (uint32_t)((uint64_t)site >> 32), 0u, 0u };
    uint32_t r[4];
    aho_philox4x32_10(ctr, key, r);
    if (kind == 0) {
        double th = AHO_TWO_PI * aho_u53(r[0], r[1]);
        *re = p->sigma * cos(th);
        *im = p->sigma * sin(th);
    } else {
        double u1 = aho_u53(r[0], r[1]) + 1.0 / 18014398509481984.0; /* + 2^-54 */
        double u2 = aho_u53(r[2], r[3]);
        double rho = sqrt(-2.0 * log(u1));
        double amp = (p->sigma / sqrt(2.0)) * rho;
        double th = AHO_TWO_PI * u2;
        *re = amp * cos(th);
        *im = amp * sin(th);
    }
}

void aho_ic(const aho_params* p, uint64_t seed, int32_t kind, double* f10)
{
    const int64_t N = p->N, V = N * N * N;
    memset(f10, 0, (size_t)(10 * V) * sizeof(double));
    double* phi_re = f10;
    double* phi_im = f10 + V;
    uint32_t key[2] = { (uint32_t)(seed & 0xffffffffu), (uint32_t)(seed >> 32) };
#pragma omp parallel for num_threads(aho_threads) schedule(static)
    for (int64_t site = 0; site < V; ++site) aho_ic_site(p, key, site, kind, &phi_re[site], &phi_im[site]);
}

/* The same initial condition on a WINDOW of a larger lattice: f10 is a B^3 container (B = p->N) that receives the values of
 * the sites ((x0+i) mod Nfull, (y0+j) mod Nfull, (z0+k) mod Nfull) of the Nfull^3 lattice (site index of the FULL lattice
 * keys Philox).  Used by the full-size sampled parity test: the window is then stepped as a small periodic lattice and only
 * its interior, which the wrong wrap cannot have reached after n steps (one site per step), is compared.
 * pinned by: equality with the corresponding sub-box of aho_ic on a lattice small enough to generate in full. */
void aho_ic_window(const aho_params* p, uint64_t seed, int32_t kind, int64_t Nfull, int64_t x0, int64_t y0, int64_t z0, double* f10)
{
    const int64_t B = p->N, V = B * B * B;
    memset(f10, 0, (size_t)(10 * V) * sizeof(double));
    uint32_t key[2] = { (uint32_t)(seed & 0xffffffffu), (uint32_t)(seed >> 32) };
    for (int64_t k = 0; k < B; ++k)
        for (int64_t j = 0; j < B; ++j)
            for (int64_t i = 0; i < B; ++i) {
                const int64_t x = ((x0 + i) % Nfull + Nfull) % Nfull, y = ((y0 + j) % Nfull + Nfull) % Nfull, z = ((z0 + k) % Nfull + Nfull) % Nfull;
                const int64_t site = x + Nfull * (y + Nfull * z), w = i + B * (j + B * k);
                aho_ic_site(p, key, site, kind, &f10[w], &f10[V + w]);
            }
}

/* ----------------------------------------------------------------------------------------------
 * Scale factor and running couplings (a ~ eta^m ; Eq. 8).
 * -------------------------------------------------------------------------------------------- */
static double aho_a(const aho_params* p, double tau) { return pow(tau / p->tau_ref, p->m); }
/* s of Eq. 8 at conformal time tau: the constant p->s, or the piecewise-linear schedule (R23: the paper's runs "with core
 * growth" change s during the run, L66-70, but do not give the schedule) */
static double aho_s(const aho_params* p, double tau)
{
    if (p->ns <= 0) return p->s;
    if (tau <= p->sched_tau[0]) return p->sched_s[0];
    for (int32_t k = 1; k < p->ns; ++k)
        if (tau <= p->sched_tau[k]) {
            const double w = (tau - p->sched_tau[k - 1]) / (p->sched_tau[k] - p->sched_tau[k - 1]);
            return p->sched_s[k - 1] + w * (p->sched_s[k] - p->sched_s[k - 1]);
        }
    return p->sched_s[p->ns - 1];
}
static double aho_e(const aho_params* p, double a, double tau) { return p->e0 * pow(a, aho_s(p, tau) - 1.0); }
static double aho_lambda(const aho_params* p, double a, double tau) { return p->lambda0 * pow(a, 2.0 * (aho_s(p, tau) - 1.0)); }
static double aho_tau(const aho_params* p, int64_t n) { return p->tau0 + (double)n * p->dt; }

/* ----------------------------------------------------------------------------------------------
 * The six coefficients of Eqs. 4-5 for the step n -> n+1, read off the
 * equations as printed:
 *   c[0] = c1 = (a_{n-1/2}/a_{n+1/2})^2                      damping of Pi       (Eq. 4, 1st term)
 *   c[1] = c2 = (dt/dx^2) (a_n/a_{n+1/2})^2                  Laplacian           (Eq. 4, 3rd term)
 *   c[2] = c3 = dt (a_n^2/a_{n+1/2})^2 lambda_n / 2          Higgs force         (Eq. 4, 2nd term)
 *   c[3] = d1 = (e_{n+1/2}/e_{n-1/2})^2                      damping of E        (Eq. 5, 1st term)
 *   c[4] = d2 = 2 dt a_n^2 e_{n+1/2}^2                       gauge current       (Eq. 5, 2nd term)
 *   c[5] = d3 = (dt/dx^2) (e_{n+1/2}/e_n)^2                  plaquette curl      (Eq. 5, 3rd term)
 * pinned by: homogeneous-mode scalar recurrence (P9), Gauss's law for several (m,s) (P1),
 * dispersion relation (P8), closed forms at s=1 (d1 = 1, d3 = dt/dx^2) and m=0.
 * -------------------------------------------------------------------------------------------- */
void aho_coeffs(const aho_params* p, int64_t n, double c[6])
{
    const double tau = aho_tau(p, n);
    const double am = aho_a(p, tau - 0.5 * p->dt);
    const double a0 = aho_a(p, tau);
    const double ap = aho_a(p, tau + 0.5 * p->dt);
    const double em = aho_e(p, am, tau - 0.5 * p->dt), e0 = aho_e(p, a0, tau), ep = aho_e(p, ap, tau + 0.5 * p->dt);
    const double lam0 = aho_lambda(p, a0, tau);
    const double idx2 = 1.0 / (p->dx * p->dx);
    c[0] = (am / ap) * (am / ap);
    c[1] = p->dt * idx2 * (a0 / ap) * (a0 / ap);
    c[2] = p->dt * (a0 * a0 / ap) * (a0 * a0 / ap) * lam0 * 0.5;
    c[3] = (ep / em) * (ep / em);
    c[4] = 2.0 * p->dt * a0 * a0 * ep * ep;
    c[5] = p->dt * idx2 * (ep / e0) * (ep / e0);
}

/* periodic neighbour index: site (x,y,z) displaced by d = +-1 along direction dir */
static int64_t aho_nb(int64_t N, int64_t x, int64_t y, int64_t z, int dir, int d)
{
    if (dir == 0) x = (x + d + N) % N;
    if (dir == 1) y = (y + d + N) % N;
    if (dir == 2) z = (z + d + N) % N;
    return x + N * (y + N * z);
}

/* Plaquette angle Xi_ij at the site with coordinates (x,y,z)  (Eq. 3):
 *   Xi_ij^x = theta_i^x + theta_j^{x+k_i} - theta_i^{x+k_j} - theta_j^x                          */
static double aho_plaq(int64_t N, const double* const th[3], int64_t x, int64_t y, int64_t z, int i, int j)
{
    const int64_t s0 = x + N * (y + N * z);
    const int64_t si = aho_nb(N, x, y, z, i, +1);
    const int64_t sj = aho_nb(N, x, y, z, j, +1);
    return th[i][s0] + th[j][si] - th[i][sj] - th[j][s0];
}

/* ----------------------------------------------------------------------------------------------
 * One leapfrog step n -> n+1 (Eqs. 4-7), in place on f10.
 *   kick  (Eq. 4): Pi  <- c1 Pi  - c3 (|phi|^2 - sigma^2) phi + c2 sum_j [U_j^x phi^{x+k_j} - 2 phi^x + conj(U_j^{x-k_j}) phi^{x-k_j}]
 *   kick  (Eq. 5): eps_i <- d1 eps_i + d2 q Im[conj(phi^x) U_i^x phi^{x+k_i}] - d3 sum_{j!=i} [sin Xi_ij^x - sin Xi_ij^{x-k_j}]
 *   drift (Eqs. 6-7): phi <- phi + dt Pi ,  theta_i <- theta_i + dt eps_i   (freshly kicked Pi, eps)
 * Both kicks read only level-n fields, so the kicks are done for all sites first (Pi, eps are
 * site/link local), then the drift in a second sweep.  U_j^x = cos(theta_j^x) - i q sin(theta_j^x).
 * (Eqs. 4-5 as printed are the q = -1 form; R1.)
 * pinned by: brute-force per-term evaluation on 4^3 (P3), force = -dH/dfield (P2), vacuum and
 * pure gauge (P4), energy (P5), time reversal (P6), lattice symmetries (P7), dispersion (P8),
 * homogeneous mode (P9), Gauss's law (P1), charge conjugation (P12).
 * -------------------------------------------------------------------------------------------- */
static void aho_step_once(const aho_params* p, double* f10, int64_t n)
{
    const int64_t N = p->N, V = N * N * N;
    const double q = (double)p->q;
    double* phr = f10;           double* phi_ = f10 + V;
    double* pir = f10 + 2 * V;   double* pii = f10 + 3 * V;
    double* th[3]  = { f10 + 4 * V, f10 + 5 * V, f10 + 6 * V };
    double* eps[3] = { f10 + 7 * V, f10 + 8 * V, f10 + 9 * V };
    const double* const thc[3] = { th[0], th[1], th[2] };
    double c[6];
    aho_coeffs(p, n, c);
    const double c1 = c[0], c2 = c[1], c3 = c[2], d1 = c[3], d2 = c[4], d3 = c[5];
    const double sig2 = p->sigma * p->sigma;

#pragma omp parallel for num_threads(aho_threads) schedule(static)
    for (int64_t z = 0; z < N; ++z)
    for (int64_t y = 0; y < N; ++y)
    for (int64_t x = 0; x < N; ++x) {
        const int64_t s0 = x + N * (y + N * z);
        const double fr = phr[s0], fi = phi_[s0];
        /* --- Eq. 4: covariant Laplacian ------------------------------------------------------ */
        double lap_re = 0.0, lap_im = 0.0;
        for (int j = 0; j < 3; ++j) {
            const int64_t sp = aho_nb(N, x, y, z, j, +1);
            const int64_t sm = aho_nb(N, x, y, z, j, -1);
            /* U_j^x phi^{x+k_j},  U = cos - i q sin */
            const double cu = cos(th[j][s0]), su = sin(th[j][s0]);
            const double fwd_re = cu * phr[sp] + q * su * phi_[sp];
            const double fwd_im = cu * phi_[sp] - q * su * phr[sp];
            /* conj(U_j^{x-k_j}) phi^{x-k_j},  conj(U) = cos + i q sin */
            const double cb = cos(th[j][sm]), sb = sin(th[j][sm]);
            const double bwd_re = cb * phr[sm] - q * sb * phi_[sm];
            const double bwd_im = cb * phi_[sm] + q * sb * phr[sm];
            lap_re += fwd_re - 2.0 * fr + bwd_re;
            lap_im += fwd_im - 2.0 * fi + bwd_im;
        }
        const double mod2 = fr * fr + fi * fi;
        const double new_pir = c1 * pir[s0] - c3 * (mod2 - sig2) * fr + c2 * lap_re;
        const double new_pii = c1 * pii[s0] - c3 * (mod2 - sig2) * fi + c2 * lap_im;
        /* --- Eq. 5: current and plaquette curl, for each link direction i -------------------- */
        double new_eps[3];
        for (int i = 0; i < 3; ++i) {
            const int64_t sp = aho_nb(N, x, y, z, i, +1);
            const double cu = cos(th[i][s0]), su = sin(th[i][s0]);
            const double fwd_re = cu * phr[sp] + q * su * phi_[sp];
            const double fwd_im = cu * phi_[sp] - q * su * phr[sp];
            /* Im[conj(phi^x) (U phi^{x+k_i})] */
            const double cur = q * (fr * fwd_im - fi * fwd_re);
            double curl = 0.0;
            for (int j = 0; j < 3; ++j) {
                if (j == i) continue;
                int64_t xm = x, ym = y, zm = z;
                if (j == 0) xm = (x - 1 + N) % N;
                if (j == 1) ym = (y - 1 + N) % N;
                if (j == 2) zm = (z - 1 + N) % N;
                curl += sin(aho_plaq(N, thc, x, y, z, i, j)) - sin(aho_plaq(N, thc, xm, ym, zm, i, j));
            }
            new_eps[i] = d1 * eps[i][s0] + d2 * cur - d3 * curl;
        }
        /* Pi and eps are local: overwrite now; phi and theta stay at level n until the 2nd sweep */
        pir[s0] = new_pir; pii[s0] = new_pii;
        eps[0][s0] = new_eps[0]; eps[1][s0] = new_eps[1]; eps[2][s0] = new_eps[2];
    }
    /* --- Eqs. 6-7: drift -------------------------------------------------------------------- */
#pragma omp parallel for num_threads(aho_threads) schedule(static)
    for (int64_t s0 = 0; s0 < V; ++s0) {
        phr[s0]  += p->dt * pir[s0];
        phi_[s0] += p->dt * pii[s0];
        th[0][s0] += p->dt * eps[0][s0];
        th[1][s0] += p->dt * eps[1][s0];
        th[2][s0] += p->dt * eps[2][s0];
    }
}

/* nsteps leapfrog steps starting from the snapshot after n0 steps */
void aho_step(const aho_params* p, double* f10, int64_t n0, int32_t nsteps)
{
    for (int32_t k = 0; k < nsteps; ++k) aho_step_once(p, f10, n0 + k);
}

/* ----------------------------------------------------------------------------------------------
 * Winding (Eq. 11; Kajantie et al. 1998).  With arg^x = atan2(phi_im, phi_re):
 *   delta_i^x = arg^{x+k_i} - arg^x - q theta_i^x
 *   n_i^x     = rint(delta_i^x * INV_2PI)                   ("[...]_pi": multiples of 2 pi, R7)
 *   Y_i^x     = delta_i^x - 2 pi n_i^x + q theta_i^x = (arg^{x+k_i} - arg^x) - 2 pi n_i^x
 *   W_ij^x    = (Y_i^x + Y_j^{x+k_i} - Y_i^{x+k_j} - Y_j^x) / 2 pi
 *             = -(n_i^x + n_j^{x+k_i} - n_i^{x+k_j} - n_j^x)   since the arg differences telescope,
 * an exact integer, evaluated in integer arithmetic for (i,j) in {(0,1),(0,2),(1,2)}.
 * W3 (optional, may be NULL) receives the three W arrays, plane ij-major: W3[p*N^3 + site].
 * (Eq. 11 as printed is the q = -1 form; R1.)
 * pinned by: hand-built string-antistring pair (P10: exactly 2N pierced plaquettes), literal
 * floating-point Eq. 11 (P13), random lattice gauge transformation (P11), 1/3 pierced fraction of
 * the random-phase IC (P15).
 * -------------------------------------------------------------------------------------------- */
void aho_winding(const aho_params* p, const double* f10, int32_t* W3, uint64_t* n_pierced, uint64_t* sum_abs_w)
{
    const int64_t N = p->N, V = N * N * N;
    const double q = (double)p->q;
    const double* phr = f10;
    const double* phi_ = f10 + V;
    const double* th[3] = { f10 + 4 * V, f10 + 5 * V, f10 + 6 * V };
    double* arg = (double*)malloc((size_t)V * sizeof(double));
    int32_t* nl = (int32_t*)malloc((size_t)(3 * V) * sizeof(int32_t));
#pragma omp parallel for num_threads(aho_threads) schedule(static)
    for (int64_t s0 = 0; s0 < V; ++s0) arg[s0] = atan2(phi_[s0], phr[s0]);
#pragma omp parallel for num_threads(aho_threads) schedule(static)
    for (int64_t z = 0; z < N; ++z)
    for (int64_t y = 0; y < N; ++y)
    for (int64_t x = 0; x < N; ++x) {
        const int64_t s0 = x + N * (y + N * z);
        for (int i = 0; i < 3; ++i) {
            const int64_t sp = aho_nb(N, x, y, z, i, +1);
            const double delta = arg[sp] - arg[s0] - q * th[i][s0];
            nl[i * V + s0] = (int32_t)rint(delta * AHO_INV_2PI);
        }
    }
    static const int PI_[3] = { 0, 0, 1 }, PJ_[3] = { 1, 2, 2 };
    uint64_t cnt = 0, tot = 0;
    for (int pl = 0; pl < 3; ++pl) {
        const int i = PI_[pl], j = PJ_[pl];
#pragma omp parallel for num_threads(aho_threads) schedule(static) reduction(+ : cnt, tot)   /* integer sums: any order */
        for (int64_t z = 0; z < N; ++z)
        for (int64_t y = 0; y < N; ++y)
        for (int64_t x = 0; x < N; ++x) {
            const int64_t s0 = x + N * (y + N * z);
            const int64_t si = aho_nb(N, x, y, z, i, +1);
            const int64_t sj = aho_nb(N, x, y, z, j, +1);
            const int32_t W = -(nl[i * V + s0] + nl[j * V + si] - nl[i * V + sj] - nl[j * V + s0]);
            if (W3) W3[pl * V + s0] = W;
            if (W != 0) ++cnt;
            tot += (uint64_t)(W < 0 ? -W : W);
        }
    }
    free(arg); free(nl);
    *n_pierced = cnt;
    *sum_abs_w = tot;
}

/* ----------------------------------------------------------------------------------------------
 * Per-site Lagrangian density (Eq. 2) and the pieces of Eq. 10 (L83), on the
 * snapshot after n steps, a = a(tau_n) (R11):
 *   G^x   = (1/dx^2) sum_i |U_i^x phi^{x+k_i} - phi^x|^2                                 (|D phi|^2)
 *   K^x   = |Pi^x|^2
 *   Vp^x  = (a^2 lambda(a)/4) (|phi^x|^2 - sigma^2)^2
 *   El^x  = sum_i eps_i^2 / (2 e(a)^2 a^2 dx^2),  Bm^x = sum_i sum_{j!=i} (1 - cos Xi_ij^x) / (2 e(a)^2 a^2 dx^4)
 *   Lag^x = c_E El - c_B Bm + K - G - Vp          (c_E = c_B = 1: the Lagrangian whose variation is Eqs. 4-7)
 * out6 = {K, G, Lag, Vp, El, Bm}.  Vp is also the weight of the potential-weighted estimator <v^2>_V (L86);
 * a constant factor on a weight drops out of R, so its a^2 lambda(a)/4 prefactor is immaterial there.
 * El and Bm (always with unit factors) are the electric and magnetic energy densities of the equation-of-state
 * estimator, Eq. 12.
 * -------------------------------------------------------------------------------------------- */
static void aho_site_lagrangian(const aho_params* p, const double* f10, double a, double tau,
                                int64_t x, int64_t y, int64_t z, double out6[6])
{
    const int64_t N = p->N, V = N * N * N;
    const double q = (double)p->q;
    const double* phr = f10;           const double* phi_ = f10 + V;
    const double* pir = f10 + 2 * V;   const double* pii = f10 + 3 * V;
    const double* const th[3]  = { f10 + 4 * V, f10 + 5 * V, f10 + 6 * V };
    const double* const eps[3] = { f10 + 7 * V, f10 + 8 * V, f10 + 9 * V };
    const int64_t s0 = x + N * (y + N * z);
    const double idx2 = 1.0 / (p->dx * p->dx);
    const double ea = aho_e(p, a, tau), la = aho_lambda(p, a, tau);
    const double fr = phr[s0], fi = phi_[s0];
    double G = 0.0;
    for (int i = 0; i < 3; ++i) {
        const int64_t sp = aho_nb(N, x, y, z, i, +1);
        const double cu = cos(th[i][s0]), su = sin(th[i][s0]);
        const double dre = cu * phr[sp] + q * su * phi_[sp] - fr;
        const double dim = cu * phi_[sp] - q * su * phr[sp] - fi;
        G += dre * dre + dim * dim;
    }
    G *= idx2;
    const double K = pir[s0] * pir[s0] + pii[s0] * pii[s0];
    const double dm = fr * fr + fi * fi - p->sigma * p->sigma;
    const double Vp = 0.25 * a * a * la * dm * dm;
    double e2 = 0.0, mag = 0.0;
    for (int i = 0; i < 3; ++i) {
        e2 += eps[i][s0] * eps[i][s0];
        for (int j = 0; j < 3; ++j) {
            if (j == i) continue;
            mag += 1.0 - cos(aho_plaq(N, th, x, y, z, i, j));   /* ordered pairs (R12) */
        }
    }
    const double gn = 1.0 / (2.0 * ea * ea * a * a * p->dx * p->dx);
    const double El = gn * e2, Bm = gn * idx2 * mag;
    out6[0] = K; out6[1] = G; out6[2] = (p->c_E * El - p->c_B * Bm) + K - G - Vp; out6[3] = Vp; out6[4] = El; out6[5] = Bm;
}

/* ----------------------------------------------------------------------------------------------
 * Diagnostics on the snapshot after n steps.
 *   winding                       : aho_winding above; L = (pi/6) dx n_pierced, xi = sqrt((N dx)^3/L) (L88-93)
 *   <v^2>_L = 2R/(1+R), R = sum K*Lag / sum G*Lag                                  (Eqs. 9-10)
 *   <v^2>_V : the same with the potential Vp as the weight (L86: "two different weight functions")
 *   xi_L = sqrt(-mu / mean Lag) (Eq. 9); the paper does not give mu: mu = 2 pi sigma^2, the Bogomolnyi
 *          string tension at lambda = 2 e^2 (the paper's couplings, L72) -- a labelled assumption (R20)
 *   <v^2>_omega = (1 + 3 p_L / rho_L) / 2 (Eq. 12), p_L / rho_L = sum p Lag / sum rho Lag with the energy density and
 *          pressure of the model -- the paper takes them from Hindmarsh et al. (2017a), which is not in the container; these
 *          are the standard ones, a labelled assumption (R22):
 *            rho = K + G + Vp + El + Bm,   p = K - G/3 - Vp + (El + Bm)/3
 *   Gauss residual (L72, L181; derived from Eqs. 4-7, R4), a_h = a(tau_n - dt/2):
 *     g^x = sum_i (eps_i^x - eps_i^{x-k_i}) - 2 q dx^2 e0^2 a_h^(2s) Im[conj(phi^x) Pi^x]
 * Sums are accumulated in fp64: x-fastest within a z-plane, then the plane sums in z order.
 * pinned by: gauge invariance of W, <v^2>, g (P11); Gauss at roundoff after k steps for several
 * (m,s) (P1) -- the residual uses only this function's formula and the step's output, a dropped
 * factor or wrong a-level in either shows up as an O(1) residual; independent numpy evaluation of
 * Eq. 2 / Eq. 10 in tests (P17); H built from the same K, G, Vp pieces conserves energy (P5).
 * -------------------------------------------------------------------------------------------- */
void aho_diag_compute(const aho_params* p, const double* f10, int64_t n, aho_diag* out)
{
    const int64_t N = p->N, V = N * N * N;
    const double q = (double)p->q;
    const double* phr = f10;           const double* phi_ = f10 + V;
    const double* pir = f10 + 2 * V;   const double* pii = f10 + 3 * V;
    const double* const eps[3] = { f10 + 7 * V, f10 + 8 * V, f10 + 9 * V };
    memset(out, 0, sizeof(*out));

    for (int64_t k = 0; k < 10 * V; ++k) if (!isfinite(f10[k])) { out->nonfinite = 1; break; }

    aho_winding(p, f10, NULL, &out->n_pierced, &out->sum_abs_w);
    out->L = (M_PI / 6.0) * p->dx * (double)out->n_pierced;
    {
        const double box = (double)N * p->dx;
        out->xi = out->n_pierced ? sqrt(box * box * box / out->L) : INFINITY;
    }

    const double tau = aho_tau(p, n);
    const double a = aho_a(p, tau);
    const double ah = aho_a(p, tau - 0.5 * p->dt);
    const double eh = aho_e(p, ah, tau - 0.5 * p->dt);   /* e(a_h)^2 a_h^2 = e0^2 a_h^(2s) for a constant s */
    const double grhs = 2.0 * q * p->dx * p->dx * eh * eh * ah * ah;
    /* per z-plane sums in x-fastest order (planes are independent), then the planes added in z order */
    double* plane = (double*)malloc((size_t)N * 9 * sizeof(double));
#pragma omp parallel for num_threads(aho_threads) schedule(static)
    for (int64_t z = 0; z < N; ++z) {
        double num = 0.0, den = 0.0, lsum = 0.0, gmax = 0.0, rhs2 = 0.0, vnum = 0.0, vden = 0.0, wnum = 0.0, wden = 0.0;
        for (int64_t y = 0; y < N; ++y)
        for (int64_t x = 0; x < N; ++x) {
            const int64_t s0 = x + N * (y + N * z);
            double kgl[6];
            aho_site_lagrangian(p, f10, a, tau, x, y, z, kgl);
            num  += kgl[0] * kgl[2];
            den  += kgl[1] * kgl[2];
            lsum += kgl[2];
            vnum += kgl[0] * kgl[3];
            vden += kgl[1] * kgl[3];
            {   /* Eq. 12: pressure and energy density, weighted with the Lagrangian */
                const double rho = kgl[0] + kgl[1] + kgl[3] + kgl[4] + kgl[5];
                const double prs = kgl[0] - kgl[1] / 3.0 - kgl[3] + (kgl[4] + kgl[5]) / 3.0;
                wnum += prs * kgl[2];
                wden += rho * kgl[2];
            }
            double div = 0.0;
            for (int i = 0; i < 3; ++i) div += eps[i][s0] - eps[i][aho_nb(N, x, y, z, i, -1)];
            const double rhs = grhs * (phr[s0] * pii[s0] - phi_[s0] * pir[s0]);
            const double g = fabs(div - rhs);
            if (g > gmax || g != g) gmax = g;
            rhs2 += rhs * rhs;
        }
        double* o = plane + 9 * z;
        o[0] = num; o[1] = den; o[2] = lsum; o[3] = gmax; o[4] = rhs2; o[5] = vnum; o[6] = vden; o[7] = wnum; o[8] = wden;
    }
    double num = 0.0, den = 0.0, lsum = 0.0, gmax = 0.0, rhs2 = 0.0, vnum = 0.0, vden = 0.0, wnum = 0.0, wden = 0.0;
    for (int64_t z = 0; z < N; ++z) {
        const double* o = plane + 9 * z;
        num += o[0]; den += o[1]; lsum += o[2]; rhs2 += o[4]; vnum += o[5]; vden += o[6]; wnum += o[7]; wden += o[8];
        if (o[3] > gmax || o[3] != o[3]) gmax = o[3];
    }
    free(plane);
    out->v2_num = num;
    out->v2_den = den;
    {
        const double R = num / den;
        out->v2 = 2.0 * R / (1.0 + R);
    }
    out->mean_lagrangian = lsum / (double)V;
    out->v2v_num = vnum;
    out->v2v_den = vden;
    {
        const double R = vnum / vden;
        out->v2_V = 2.0 * R / (1.0 + R);
    }
    out->xi_L = sqrt(-(AHO_TWO_PI * p->sigma * p->sigma) / out->mean_lagrangian);
    out->eos_num = wnum;
    out->eos_den = wden;
    out->v2_omega = 0.5 * (1.0 + 3.0 * wnum / wden);
    out->gauss_max = gmax;
    out->gauss_rhs_rms = sqrt(rhs2 / (double)V);
}

/* per-site arrays K, G, Lag and (if not NULL) Vp (each N^3) for tests that re-evaluate Eq. 2 independently */
void aho_site_fields4(const aho_params* p, const double* f10, int64_t n, double* K, double* G, double* Lag, double* Vp)
{
    const int64_t N = p->N;
    const double tau = aho_tau(p, n);
    const double a = aho_a(p, tau);
#pragma omp parallel for num_threads(aho_threads) schedule(static)
    for (int64_t z = 0; z < N; ++z)
    for (int64_t y = 0; y < N; ++y)
    for (int64_t x = 0; x < N; ++x) {
        double kgl[6];
        aho_site_lagrangian(p, f10, a, tau, x, y, z, kgl);
        const int64_t s0 = x + N * (y + N * z);
        K[s0] = kgl[0]; G[s0] = kgl[1]; Lag[s0] = kgl[2];
        if (Vp) Vp[s0] = kgl[3];
    }
}
/* the electric and magnetic energy densities El, Bm (each N^3) as well */
void aho_site_fields6(const aho_params* p, const double* f10, int64_t n, double* K, double* G, double* Lag, double* Vp, double* El, double* Bm)
{
    const int64_t N = p->N;
    const double tau = aho_tau(p, n);
    const double a = aho_a(p, tau);
#pragma omp parallel for num_threads(aho_threads) schedule(static)
    for (int64_t z = 0; z < N; ++z)
    for (int64_t y = 0; y < N; ++y)
    for (int64_t x = 0; x < N; ++x) {
        double kgl[6];
        aho_site_lagrangian(p, f10, a, tau, x, y, z, kgl);
        const int64_t s0 = x + N * (y + N * z);
        K[s0] = kgl[0]; G[s0] = kgl[1]; Lag[s0] = kgl[2]; Vp[s0] = kgl[3]; El[s0] = kgl[4]; Bm[s0] = kgl[5];
    }
}
void aho_site_fields(const aho_params* p, const double* f10, int64_t n, double* K, double* G, double* Lag)
{
    aho_site_fields4(p, f10, n, K, G, Lag, NULL);
}

/* struct sizes, so the ctypes mirror in ahs_oracle.py can assert it matches */
int32_t aho_sizeof_params(void) { return (int32_t)sizeof(aho_params); }
int32_t aho_sizeof_diag(void) { return (int32_t)sizeof(aho_diag); }
