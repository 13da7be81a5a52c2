/*
 * ahs.h -- C ABI of libahs: the data-parallel hot path of arXiv 1809.00995 (Correia & Martins,
 * "Abelian-Higgs Cosmic String Evolution with CUDA") on one NVIDIA B200 (sm_100a).
 *
 * What the library computes (citations are PAPER.md line numbers; "R<n>" = readings in DESIGN.md):
 *   - the damped staggered-leapfrog update, Eqs. 4-7 (L55-L62), of a complex scalar phi and its
 *     momentum Pi on the sites and of the U(1) link angles theta_i and their conjugates eps_i on the
 *     links of a periodic N^3 comoving lattice, with a(tau) = (tau/tau_ref)^m (L224, R3) and the
 *     core-width parameter s of Eq. 8 (L68): e(a) = e0 a^(s-1), lambda(a) = lambda0 a^(2(s-1));
 *   - the network diagnostics: plaquette winding, Eq. 11 (L88-L93), giving the string length
 *     L = (pi/6) dx n_pierced and xi = sqrt((N dx)^3 / L); the Lagrangian-weighted mean square velocity,
 *     Eqs. 9-10 with the weight of Eq. 2 (L40, L78-L86); and the residual of the discrete Gauss law
 *     (L72, L181; R4).
 *
 * Variables.  The stored "A" and "E" are the paper's rescaled link variables (L44, R5):
 *     theta_i = e0 * dx * A_i   (dimensionless link angle, U_i^x = exp(-i theta_i^x), R1)
 *     eps_i   = d theta_i / d eta.
 * A field snapshot "after n steps" is { phi^n, theta^n at tau_n = tau0 + n dt ; Pi^(n-1/2), eps^(n-1/2) }.
 * Fields cross this boundary as 10 contiguous arrays of N^3 values in the order
 *     phi_re, phi_im, Pi_re, Pi_im, theta_0, theta_1, theta_2, eps_0, eps_1, eps_2
 * with site index  x + N*(y + N*z)  (x fastest; direction 0,1,2 = x,y,z; theta_i^x sits on the link
 * from x to x + k_i).
 *
 * Pointers.  Every pointer argument says HOST or DEVICE.  The caller owns every host pointer it passes.
 * The library owns the device memory it allocates; if ahs_params.device_buffer is given the caller owns
 * it and frees it after ahs_destroy.  All work of a handle is issued on the handle's CUDA stream;
 * ahs_step is asynchronous, every function that returns data to the host synchronises that stream.
 * A handle is not thread-safe; distinct handles are independent (replicas).
 *
 * Devices.  A handle belongs to the device that was current when it was created (a caller-supplied device_buffer must
 * live there).  Every later call makes that device current for its own duration and restores the caller's, so one host
 * thread can drive handles on several GPUs without calling cudaSetDevice itself.
 *
 * Errors.  Functions returning int return AHS_OK (0) or a negative code; ahs_last_error() returns a
 * thread-local, statically stored, human readable message for the last failure on the calling thread.
 * There is no CPU fallback and no other backend: without a CUDA device every call that needs one fails
 * with AHS_ERR_CUDA.
 */
#ifndef AHS_H_
#define AHS_H_

#include <stddef.h>
#include <stdint.h>

#if defined(__GNUC__)
#define AHS_API __attribute__((visibility("default")))
#else
#define AHS_API
#endif

#ifdef __cplusplus
extern "C" {
#endif

typedef struct ahs_sim ahs_sim; /* opaque handle */

enum { AHS_OK = 0, AHS_ERR_INVALID_ARG = -1, AHS_ERR_OOM = -2, AHS_ERR_CUDA = -3, AHS_ERR_NONFINITE = -4, AHS_ERR_STATE = -5 };
enum { AHS_F32 = 0, AHS_F64 = 1 };                                   /* storage AND arithmetic type of the step */
enum { AHS_IC_RANDOM_PHASE = 0, AHS_IC_GAUSSIAN = 1, AHS_IC_NONE = 2 /* all fields zero; set them with ahs_set_fields */ };
enum { AHS_KERNEL_AUTO = 0, AHS_KERNEL_GENERIC = 1, AHS_KERNEL_MARCH = 2 };
enum { AHS_OPT_STAGING = 0, AHS_OPT_STEP_CHUNKS = 1, AHS_OPT_DIAG_CHUNKS = 2, AHS_OPT_DIAG_TRIG = 3, AHS_OPT_STEP_PDL = 4 };   /* ahs_set_option */
enum { AHS_STAGING_TENSOR = 0, AHS_STAGING_ROWS = 1 };
enum { AHS_TRIG_HARDWARE = 0, AHS_TRIG_POLYNOMIAL = 1 };
enum { AHS_EXCHANGE_STORES = 0, AHS_EXCHANGE_COPIES = 1 };           /* ahs_group_set_exchange */

/*
 * Parameters of a simulation (L36: lambda, e, sigma; L51: dx, dt; L68-70: s; L224: a ~ eta^m; L72: IC).
 *   N               lattice is N^3, periodic, 4 <= N <= 2048.  The z-marching kernels (TMA-staged tiles, the ones that run near
 *                   the HBM roofline) need N % 128 == 0 (fp32) or N % 64 == 0 (fp64) and are chosen automatically when that
 *                   holds.  Any other N runs on the one-thread-per-site kernels, which are about 6 x slower on the step and
 *                   8 x slower on the diagnostics (profiles/HISTORY.md r1); ahs_kernel_kind tells which one a handle uses.
 *   dx, dt          lattice spacing and conformal time step, > 0.
 *   lambda, e, sigma  lambda_0, e_0 of Eq. 8 and the vacuum expectation value, > 0.
 *   m               a(tau) = (tau/tau_ref)^m : 0 static, 1 radiation, 2 matter.
 *   s               Eq. 8: 0 = constant comoving core width, 1 = true equations of motion.
 *   tau0            conformal time of step 0; tau0 - dt/2 > 0 is required when m != 0.
 *   tau_ref         normalisation of a (R3); 0 means tau0, i.e. a(tau0) = 1.
 *   seed            Philox4x32-10 key (lo 32 bits, hi 32 bits); counter = (site lo, site hi, 0, 0)  (R9).
 *   precision       AHS_F32 or AHS_F64.
 *   ic_kind         AHS_IC_RANDOM_PHASE: phi = sigma exp(2 pi i u), Pi = theta = eps = 0 (L72);
 *                   AHS_IC_GAUSSIAN: re, im ~ N(0, sigma^2/2) by Box-Muller; AHS_IC_NONE: zeros.
 *   kernel          AHS_KERNEL_AUTO, or force one of the two step/diagnostics implementations.
 *   device_buffer   DEVICE pointer, optional (NULL => the library calls cudaMalloc).  Must hold
 *                   ahs_required_bytes(N, precision) bytes, 256-byte aligned (e.g. torch.empty(...).data_ptr()).
 *   stream          cudaStream_t as void*, optional (NULL => the legacy default stream).
 *   c_B             factor on the plaquette sum of Eq. 2 (L40) in the weight of <v^2>_L and in mean_lagrangian; 0 means 1, the
 *                   value consistent with Eq. 5 (R2).  Eq. 2 as printed has 1/2; it does not enter the equations of motion.
 *   c_E             factor on the electric term sum_i eps_i^2 of Eq. 2 in the same weight; 0 means 1, the value for eps = d theta /
 *                   d eta (Eq. 7, R5).  (dt/dx)^2 is what the sentence "E_i -> e dt E_i" of L44 gives when read literally (R21);
 *                   with it <v^2>_L reproduces the paper's Table 4 within two standard deviations.
 */
typedef struct {
    int32_t N;
    int32_t precision;
    int32_t ic_kind;
    int32_t kernel;
    double dx, dt, lambda, e, sigma, m, s, tau0, tau_ref;
    uint64_t seed;
    void* device_buffer;
    size_t device_buffer_bytes;
    void* stream;
    double c_B;
    double c_E;
} ahs_params;

/* Result of one diagnostics pass on the current snapshot (after `step` steps). */
typedef struct {
    int64_t step;             /* n                                                                         */
    double tau;               /* tau_n = tau0 + n dt                                                       */
    uint64_t n_pierced;       /* plaquettes with W != 0, Eq. 11 (L88-93), bit-exact integer (fp32 lattices on the
                                 z-marching kernel: for |phi_re|, |phi_im| < 2^126; beyond, the sums overflow too) */
    uint64_t sum_abs_w;       /* sum |W| over the 3 N^3 plaquettes                                         */
    double L;                 /* (pi/6) dx n_pierced (L93)                                                 */
    double xi;                /* sqrt((N dx)^3 / L); +inf if n_pierced == 0                                */
    double v2_num;            /* sum_x |Pi|^2 Lag^x     (Eq. 10, weight = Eq. 2 with c_B = 1, R2)          */
    double v2_den;            /* sum_x |D phi|^2 Lag^x                                                     */
    double v2;                /* 2R/(1+R), R = v2_num / v2_den (Eq. 9): <v^2>_L.  NOT validated against the paper's
                                 Table 4: with the weight that is consistent with Eqs. 4-7 (c_B = c_E = 1) it comes out
                                 0.05 below the paper's value in both eras, and no reading of the printed Eq. 2 reproduces
                                 all of the paper's Lagrangian-weighted columns.  v2_V and v2_omega
                                 below agree with Table 4 within two standard deviations                                   */
    double mean_lagrangian;   /* sum_x Lag^x / N^3                                                         */
    double gauss_max;         /* max_x |sum_i (eps_i^x - eps_i^{x-k_i}) - 2 dx^2 e0^2 a_h^(2s) Im[conj(phi) Pi]|,
                                 a_h = a(tau_n - dt/2)  (R4)                                               */
    double gauss_rhs_rms;     /* rms_x of the second term: the scale gauss_max is to be compared with      */
    int32_t nonfinite;        /* 1 if any stored field value is NaN or +-inf (finite values whose products
                                 overflow the storage type make the sums non-finite but do not set this)   */
    int32_t reserved;
    double v2v_num;           /* sum_x |Pi|^2 Vp^x, Vp = (a^2 lambda(a)/4)(|phi|^2 - sigma^2)^2: Eq. 10 with the
                                 potential as the weight (L86, "two different weight functions")             */
    double v2v_den;           /* sum_x |D phi|^2 Vp^x                                                      */
    double v2_V;              /* 2R/(1+R), R = v2v_num / v2v_den: <v^2>_V (Eq. 9)                          */
    double xi_L;              /* sqrt(-mu / mean_lagrangian), Eq. 9 (L78), with mu = 2 pi sigma^2 -- the paper
                                 does not state mu; this is the Bogomolnyi tension at lambda = 2 e^2 (R20).
                                 NaN when mean_lagrangian >= 0                                              */
    double eos_num;           /* sum_x p^x Lag^x,   p = K - G/3 - Vp + (El + Bm)/3     (Eq. 12; the pressure and   */
    double eos_den;           /* sum_x rho^x Lag^x, rho = K + G + Vp + El + Bm          energy density of the model, R22:  */
    double v2_omega;          /* (1 + 3 eos_num / eos_den) / 2: <v^2>_omega             K = |Pi|^2, G = |D phi|^2, El / Bm the
                                 electric / magnetic terms of Eq. 2 with unit factors; the paper takes p, rho from a
                                 reference that is not reproduced in it, so these definitions are a labelled assumption)   */
} ahs_diag;

/* Bytes of device memory a simulation needs: 15 arrays of N^3 values (10 live + the phi', theta' shadow
 * buffers of the double-buffered drift) plus reduction scratch.  0 if N or precision is invalid. */
AHS_API size_t ahs_required_bytes(int32_t N, int32_t precision);

/* north_star signature: fp32, random-phase IC (L72), a = (tau/tau0)^m, default stream, library-owned
 * memory on the current device.  Returns NULL on failure (see ahs_last_error). */
AHS_API ahs_sim* ahs_create(int32_t N, double dx, double dt, double lambda, double e, double sigma,
                    double m, double s, double tau0, uint64_t seed);

/* General constructor.  params: HOST pointer.  Returns NULL on failure. */
AHS_API ahs_sim* ahs_create_ex(const ahs_params* params);

/* n >= 0 leapfrog steps (Eqs. 4-7), one fused kernel launch per step, asynchronous on the handle's
 * stream; the six coefficients of Eqs. 4-5 are computed on the host in fp64 from tau_n and passed as
 * kernel arguments. */
AHS_API int32_t ahs_step(ahs_sim* sim, int32_t n);

/* Diagnostics of the current snapshot.  L, v2, gauss: HOST pointers, any may be NULL.
 * L = (pi/6) dx n_pierced; v2 = <v^2>_L; gauss = max |Gauss residual| (absolute).
 * Synchronises.  Returns AHS_ERR_NONFINITE (outputs still filled) if a field value is not finite. */
AHS_API int32_t ahs_diagnostics(ahs_sim* sim, double* L, double* v2, double* gauss);
AHS_API int32_t ahs_diagnostics_ex(ahs_sim* sim, ahs_diag* out /* HOST */);

/* Launch the diagnostics kernels without reading the result back (asynchronous; for timing). The result
 * is fetched by the next ahs_diagnostics_fetch.  */
AHS_API int32_t ahs_diagnostics_launch(ahs_sim* sim);
AHS_API int32_t ahs_diagnostics_fetch(ahs_sim* sim, ahs_diag* out /* HOST */);

/* Copy the snapshot to / from HOST memory as doubles: host10 holds 10*N^3 doubles in the field order above.
 * ahs_set_fields rounds to the storage precision and sets the step counter (tau = tau0 + step*dt). Synchronise. */
AHS_API int32_t ahs_get_fields(ahs_sim* sim, double* host10);
AHS_API int32_t ahs_set_fields(ahs_sim* sim, const double* host10, int64_t step);

/* The same in the storage type (float for AHS_F32, double for AHS_F64): 10*N^3 values, no conversion, one
 * cudaMemcpyAsync per field on the handle's stream followed by a synchronise. Pinned host memory makes
 * the copies run at PCIe speed. */
AHS_API int32_t ahs_get_fields_native(ahs_sim* sim, void* host10);
AHS_API int32_t ahs_set_fields_native(ahs_sim* sim, const void* host10, int64_t step);
/* The same upload without the final synchronise: the ten copies are enqueued on the handle's stream and the call returns; later
 * work of the handle (ahs_step, diagnostics) is ordered behind them.  host10 (HOST, pinned for a truly asynchronous copy) must stay
 * valid and unchanged until a synchronising call of this handle has returned.  With two handles on two streams the upload of one
 * state overlaps the evolution of the other (bench.py's end-to-end leg). */
AHS_API int32_t ahs_set_fields_native_async(ahs_sim* sim, const void* host10, int64_t step);

/* DEVICE pointer to live field k (0..9, order above) in the storage type; valid until the next ahs_step
 * (phi and theta alternate between two buffers).  For zero-copy views from PyTorch. */
AHS_API int32_t ahs_field_device_ptr(ahs_sim* sim, int32_t k, void** dev_ptr /* HOST pointer to a DEVICE pointer */);

/* Counters: step n, tau_n, and the number of kernels launched by this handle so far. */
AHS_API int32_t ahs_get_state(ahs_sim* sim, int64_t* step, double* tau, int64_t* kernel_launches);

/* Which implementation the handle uses: AHS_KERNEL_GENERIC or AHS_KERNEL_MARCH. */
AHS_API int32_t ahs_kernel_kind(ahs_sim* sim);

/* Tuning of the z-marching kernels (no effect on the one-thread-per-site kernels; the first three have none on any result beyond
 * rounding order of the fp64 reduction, which follows the launch shape).  Takes effect at the next launch.
 *   AHS_OPT_STAGING      AHS_STAGING_TENSOR (default): halo'd tiles of the level-n fields (Eq. 4-5's phi, theta) are staged in
 *                        shared memory by tensor-map TMA copies wherever a tile does not straddle the periodic boundary in y;
 *                        AHS_STAGING_ROWS: by one bulk copy per tile row everywhere (the path tiles on that boundary always take).
 *   AHS_OPT_STEP_CHUNKS  number of z-chunks each (x, y) tile of the step march is cut into, 1..N (a slab of an ahs_group: 1..N / nslabs;
 *                        0 = the library's choice);
 *   AHS_OPT_DIAG_CHUNKS  the same for the diagnostics march.  Chunks need not divide N.
 *   AHS_OPT_DIAG_TRIG    how the diagnostics march of an fp32 lattice evaluates the sines and cosines inside the sums of Eqs. 2, 9, 10
 *                        and 12 (link phases of the gradient term, plaquette angles of the magnetic term):
 *                        AHS_TRIG_HARDWARE (default): the GPU's special-function unit, absolute error <= 4e-7 per value; the sums
 *                        then agree with an fp64 evaluation to ~1.5e-7 of their absolute sums (one fp32 rounding; measured,
 *                        DESIGN.md section 8) instead of ~1e-8;
 *                        AHS_TRIG_POLYNOMIAL: the 1-2 ulp routines the step kernel uses (the call takes ~17 % longer).
 *                        The winding (Eq. 11) and the Gauss residual do not depend on it; fp64 lattices always take the polynomials.
 *   AHS_OPT_STEP_PDL     1: the step march is launched with programmatic stream serialization -- the CTAs of step n + 1 may take the SM
 *                        slots that step n's last wave leaves free and run their set-up (barrier initialisation) there; they wait for
 *                        step n to complete before they touch global memory, so the fields are the same bit for bit.  0 (default): plain
 *                        stream order.  Matters for small lattices, where a launch lasts a fraction of a millisecond.
 * Returns AHS_ERR_INVALID_ARG for an unknown option or a value out of range. */
AHS_API int32_t ahs_set_option(ahs_sim* sim, int32_t option, int32_t value);

/* The six coefficients (c1, c2, c3, d1, d2, d3) of Eqs. 4-5 for the step n -> n+1, as the host computes
 * them. out6: HOST. */
AHS_API int32_t ahs_coefficients(ahs_sim* sim, int64_t n, double* out6);

/* A time-dependent s of Eq. 8 (L66-70: "this parameter can be controlled throughout the simulation", e.g. core growth with s < 0 and the
 * true equations, s = 1, thereafter).  The paper does not give its schedule; this one is piecewise linear in conformal time: nknots
 * strictly increasing times tau[] with values s_values[] (HOST arrays, copied), linear in between, constant outside (R23).  Every coupling
 * of Eqs. 4-5 takes s at its own time level (e at tau_n -+ dt/2 and tau_n, lambda at tau_n), and so do the weights and the Gauss residual
 * of the diagnostics.  nknots = 0 restores the constant ahs_params.s.  Takes effect at the next step / diagnostics call. */
AHS_API int32_t ahs_set_s_schedule(ahs_sim* sim, int32_t nknots, const double* tau, const double* s_values);

/* Block until all work of the handle has finished. */
AHS_API int32_t ahs_synchronize(ahs_sim* sim);

/* Free the handle and the device memory the library allocated. NULL is allowed. */
AHS_API int32_t ahs_destroy(ahs_sim* sim);

/*
 * ---- z-slab decomposition: one lattice on several handles / GPUs of this process -------------------------------------------
 * The paper's stated next step (L252-258: "extending to multiple GPUs").  The N^3 lattice is cut into nslabs slabs of N / nslabs
 * z-planes; each slab is a handle with one ghost plane below and above (15 arrays of N x N x (N/nslabs + 2) values) on
 * devices[r] (HOST array of nslabs CUDA device ordinals; NULL = the current device for all; ordinals may repeat, so the path can
 * be exercised on one GPU).  The halo exchange is part of the fused step kernel: besides its own arrays it stores the new phi,
 * theta (Eqs. 6-7) of its bottom / top plane -- and eps_2 of the top plane, which the Gauss residual of the slab above needs --
 * into the neighbouring slabs' ghost planes, through peer memory (NVLink) when they live on another GPU: 5 N^2 values per face and
 * step.  CUDA events order step n+1 of a slab behind step n of its two neighbours; nothing waits on the device.  Results are those
 * of a single handle: fields bit for bit, counts exactly, sums to the rounding order of the final reduction.
 * params: as for ahs_create_ex with device_buffer = stream = NULL and N % 128 == 0 (fp32) / N % 64 == 0 (fp64); nslabs in 1..64
 * must divide N, and a slab holds at most 2047 planes (N = 2048 needs nslabs >= 2).  Neighbouring slabs on two GPUs without peer
 * access to one another exchange that face by cudaMemcpyPeerAsync behind the step instead (5 + 5 + 1 plane copies per slab and step,
 * same values; see ahs_group_set_exchange).  One host thread drives a group.
 */
typedef struct ahs_group ahs_group;
AHS_API ahs_group* ahs_group_create(const ahs_params* params, int32_t nslabs, const int32_t* devices /* HOST, may be NULL */);
/* n steps, asynchronous like ahs_step.  If a launch or an event call fails part-way through a step, some slabs have run that step and
 * others have not: the group then refuses ahs_group_step, ahs_group_diagnostics and ahs_group_get_fields_native with AHS_ERR_STATE
 * until ahs_group_set_fields_native has set the fields again (or the group is destroyed). */
AHS_API int32_t ahs_group_step(ahs_group* group, int32_t n);
AHS_API int32_t ahs_group_diagnostics(ahs_group* group, ahs_diag* out /* HOST */);   /* every slab's pass, combined; synchronises */
/* The whole lattice in the storage type, 10 N^3 values in the field order above, gathered from / scattered to the slabs (HOST
 * pointers; ahs_group_set_fields_native also sets the step counter and fills the ghost planes).  Synchronise. */
AHS_API int32_t ahs_group_get_fields_native(ahs_group* group, void* host10);
AHS_API int32_t ahs_group_set_fields_native(ahs_group* group, const void* host10, int64_t step);
AHS_API int32_t ahs_group_synchronize(ahs_group* group);
/* How the faces travel.  AHS_EXCHANGE_STORES (default): the step kernel's own stores into the neighbours' ghost planes wherever the two
 * GPUs have peer access (always on one GPU), copies elsewhere.  AHS_EXCHANGE_COPIES: every face by cudaMemcpyPeerAsync behind the step
 * (what a pair of GPUs without peer access gets anyway; selectable so that this path can be exercised and timed on any box).  The
 * fields are the same bit for bit.  Synchronises the group.  ahs_group_exchange_faces: how many of the 2 nslabs faces go by copies. */
AHS_API int32_t ahs_group_set_exchange(ahs_group* group, int32_t mode);
AHS_API int32_t ahs_group_exchange_faces(ahs_group* group, int32_t* copied_faces /* HOST */);
AHS_API int32_t ahs_group_slab_count(ahs_group* group);
/* The handle of slab r (owned by the group: for ahs_set_option, ahs_set_s_schedule, ahs_get_state, ahs_kernel_kind, ahs_coefficients,
 * ahs_synchronize).  It is stepped, measured and its fields are read and written through the group only: ahs_step, ahs_diagnostics*,
 * ahs_get_fields* and ahs_set_fields* on it return AHS_ERR_STATE.  NULL if r is out of range. */
AHS_API ahs_sim* ahs_group_slab(ahs_group* group, int32_t r);
AHS_API int32_t ahs_group_destroy(ahs_group* group);                                 /* NULL is allowed */
/* The slab rules ahs_group_create applies, as numbers; needs no GPU (for drivers that spread slabs over processes and for the host
 * tests).  out5 (HOST, 5 ints) = { first own global plane, own planes nz, slab below, slab above (both periodic), planes allocated
 * = nz + 2 }: own planes sit at local indices 1 .. nz, local plane 0 mirrors the top own plane of the slab below, local plane nz + 1
 * the bottom own plane of the slab above.  AHS_ERR_INVALID_ARG unless nslabs in 1..64 divides N and 0 <= r < nslabs. */
AHS_API int32_t ahs_slab_layout(int32_t N, int32_t nslabs, int32_t r, int32_t* out5);

/*
 * ---- diagnostics of a snapshot the caller holds, without any allocation --------------------------------------------------------
 * Who this is for.  An evolution code that keeps its own ten field arrays on the GPU and wants the winding count (Eq. 11),
 * the <v^2> sums (Eqs. 9-10, 12) and the Gauss residual (L72, L181) of them every few steps, from a place where it may not allocate:
 *   - a production run that has sized its lattice to the last gigabyte of HBM, so that a cudaMalloc in the middle of the run can
 *     fail after hours of evolution (a handle would ask for 15 N^3 values of its own plus pinned host memory);
 *   - an analysis hook called from inside another framework's step loop (a PyTorch caching allocator that owns all free memory, a
 *     job whose device memory was partitioned up front), where cudaMalloc / cudaFree also stall every stream of the device;
 *   - a latency-critical loop that must not enter the driver's allocator at all.
 * ahs_create_ex always allocates (pinned host memory for the result, and device memory unless device_buffer is given) and copies the
 * fields into its own layout.  This call takes the caller's arrays where they are and calls no cudaMalloc, cudaMallocHost, cudaFree,
 * stream / event creation or any other allocating routine, on the host or on the device.
 *
 * Scratch.  The per-block records of the reduction (and the final record before it is read back) live in one array that is part of
 * the library image: AHS_STATIC_SCRATCH_BYTES (444.25 KiB) of device memory on EVERY GPU on which this process uses libahs, held from
 * the moment the library's code is loaded onto that GPU until the process exits, whether this function is ever called or not.  It is
 * the same one-thread-per-site kernel that AHS_KERNEL_GENERIC handles run, launched with the same shape (at most
 * AHS_STATIC_MAX_RECORDS blocks of 128 threads, one record each), so on the same snapshot it returns what such a handle returns, bit
 * for bit; it is about 8 x slower than the z-marching kernel of a handle (see N above).
 *
 * Limits.  4 <= N <= AHS_STATIC_MAX_N: the array holds a record for every block of the largest launch this kernel is given, so no
 * lattice the library accepts is too big for it; any other N, and any launch that would need more than AHS_STATIC_MAX_RECORDS
 * records, is refused with AHS_ERR_INVALID_ARG and a message naming the limit -- nothing is ever written past the array.  s is the
 * constant params->s (no s(tau) schedule).
 *
 * First call.  The first call on each device looks up the device address of the array (cudaGetSymbolAddress, with that device
 * current; this is also what makes the driver load the library's code, and with it the array, onto that GPU) and keeps it for later
 * calls.  Make that first call during set-up, before any stream capture is begun on that device.  Later calls only launch three
 * kernels (clear the result record, the site kernel, the finishing block) and copy 96 bytes back.
 *
 * Sharing.  There is ONE array per device and every call on that device uses it; it keeps whatever the last call left.  Nothing in it
 * has to start at zero for correctness -- each call writes every record before it reads it and reads only the records of its own
 * launch -- but the 96-byte result record is cleared first all the same, so that a result can never be a leftover of the call
 * before.  Two calls whose kernels can run on the GPU at the same time (different streams, different host threads, another process's
 * context does not count: it has its own copy) overwrite each other's records: the caller serialises calls per device.  A call
 * returns only after its own result has been read back, so calls made one after the other from one thread never overlap.
 *
 * Arguments.
 *   params    HOST.  Used: N, precision, dx, dt, lambda, e, sigma, m, s, tau0, tau_ref, c_B, c_E (meaning as for ahs_create_ex) and
 *             stream (the kernels and the read-back run on it; NULL = the legacy default stream).  Ignored: ic_kind, kernel, seed,
 *             device_buffer, device_buffer_bytes.
 *   fields10  HOST array of ten DEVICE pointers in the field order at the top of this file (phi_re ... eps_2), each to N^3 values of
 *             the storage type, site index x + N (y + N z), on the CURRENT device.  Read only; the caller keeps ownership and must
 *             not change them until the call returns.  Arrays taken from a handle with ahs_field_device_ptr qualify.
 *   step      n >= 0: the snapshot is { phi^n, theta^n at tau0 + n dt ; Pi^(n-1/2), eps^(n-1/2) }; sets the scale factors.
 *   out       HOST, filled as by ahs_diagnostics_ex.
 * Returns AHS_OK, AHS_ERR_NONFINITE (out still filled), AHS_ERR_INVALID_ARG (nothing launched) or AHS_ERR_CUDA.  Synchronises the
 * stream.
 */
enum { AHS_STATIC_MAX_RECORDS = 4736, AHS_STATIC_MAX_N = 2048, AHS_STATIC_SCRATCH_BYTES = 96 * (4736 + 1) + 160 /* = 454912, a multiple of 256 */ };
AHS_API int32_t ahs_diagnostics_static(const ahs_params* params /* HOST */, const void* const* fields10 /* HOST array of 10 DEVICE pointers */,
                                       int64_t step, ahs_diag* out /* HOST */);

/* Message of the last failure on this thread ("" if none). Never NULL. */
AHS_API const char* ahs_last_error(void);

/* Library version string, e.g. "ahs 0.1 sm_100a". */
AHS_API const char* ahs_version(void);

#ifdef __cplusplus
}
#endif
#endif /* AHS_H_ */
