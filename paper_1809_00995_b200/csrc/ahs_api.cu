// ahs_api.cu -- the C ABI of include/ahs.h: handle, SoA lattice store in HBM, per-step coefficient
// schedule (host, fp64), kernel dispatch, host<->device field transfer.  No torch types here: PyTorch (if the
// caller uses it) only supplies a device buffer and a stream through ahs_params.
#include <cmath>
#include <cstdarg>
#include <cstdio>
#include <cstring>
#include <new>
#include <vector>

#include "ahs_internal.cuh"

using namespace ahs;

struct ahs_sim {
    ahs_params p;
    int64_t nsites;
    size_t elem;             // sizeof storage type
    size_t array_bytes;      // bytes of one field array, rounded up to 256
    char* base;              // device buffer
    bool owns_buffer;
    cudaStream_t stream;
    int cur;                 // which (phi, theta) buffer holds level n
    int64_t step;
    int64_t launches;
    int kernel;              // AHS_KERNEL_GENERIC or AHS_KERNEL_MARCH
    DiagPartial* partials;   // device, kMaxDiagPartials records
    DiagPartial* result;     // device, 1 record
    DiagPartial* result_host;  // pinned host, 1 record
    int64_t diag_step;       // step the pending diagnostics launch refers to (-1: none)
    int device;
    DiagMaps diag_map[2];      // TMA descriptors of (phi, theta) buffer 0 / 1 for the diagnostics march
    bool diag_map_ok;
    StepMaps step_maps[2];     // the same for the step march (buffer 0 / 1 as the level-n input)
    bool step_maps_ok;
    MarchOptions opt;          // ahs_set_option
    // z-slab of an ahs_group; a whole lattice has zr = { N, 0, periodic, N } and no ghost targets
    ZRange zr;
    int z_offset;              // global plane of the first own plane
    int64_t nsites_alloc;      // N * N * zr.nz_alloc
    bool owns_stream;
    // where the step kernel also stores its bottom / top plane, per OUTPUT buffer (0 / 1): the neighbours' ghost planes
    void* ghost_lo[2][5];
    void* ghost_hi[2][5];
    void* ghost_eps2_hi;
    // A face the step kernel may NOT store through (no peer access between the two GPUs, or ahs_group_set_exchange asked for copies):
    // its ghost_* pointers above stay NULL and the same planes travel by cudaMemcpyPeerAsync behind the step, to these targets
    bool copy_lo, copy_hi;
    void* copy_lo_dst[2][5];
    void* copy_hi_dst[2][5];
    void* copy_eps2_dst;
    int lo_device, hi_device;
    // time-dependent s(tau) of Eq. 8 (ahs_set_s_schedule; R23): knots, empty = the constant p.s
    std::vector<double> sched_tau, sched_s;
};

struct SlabSpec { int nz; int z_offset; };

namespace {

thread_local char g_err[512] = "";

int fail(int code, const char* fmt, ...)
{
    va_list ap;
    va_start(ap, fmt);
    vsnprintf(g_err, sizeof(g_err), fmt, ap);
    va_end(ap);
    return code;
}

#define AHS_CUDA(call)                                                                                   \
    do {                                                                                                 \
        cudaError_t e_ = (call);                                                                         \
        if (e_ != cudaSuccess) return fail(AHS_ERR_CUDA, "%s failed: %s", #call, cudaGetErrorString(e_)); \
    } while (0)

size_t round256(size_t b) { return (b + 255) & ~(size_t)255; }

bool valid_N(int32_t N) { return N >= 4 && N <= 2048; }

size_t scratch_bytes() { return round256(sizeof(DiagPartial) * (size_t)(kMaxDiagPartials + 1)); }

template <typename T> T* slot(const ahs_sim* s, int k) { return reinterpret_cast<T*>(s->base + (size_t)k * s->array_bytes); }

// live slot of user-facing field k (0..9: phi_re, phi_im, Pi_re, Pi_im, theta_0..2, eps_0..2)
int live_slot(const ahs_sim* s, int k)
{
    const int b = s->cur ? PHI_RE1 : PHI_RE0;
    switch (k) {
        case 0: return b + 0;
        case 1: return b + 1;
        case 2: return PI_RE;
        case 3: return PI_IM;
        case 4: case 5: case 6: return b + 2 + (k - 4);
        default: return EPS0 + (k - 7);
    }
}

// ---- the scale factor and couplings (Eq. 8; R3) --------------------------------------------
double tau_of(const ahs_params& p, int64_t n) { return p.tau0 + (double)n * p.dt; }
double scale_factor(const ahs_params& p, double tau)
{
    const double tref = (p.tau_ref != 0.0) ? p.tau_ref : p.tau0;
    return std::pow(tau / tref, p.m);
}
// s of Eq. 8 at conformal time tau: constant, or piecewise linear between the knots of ahs_set_s_schedule (constant outside)
double s_of(const ahs_sim* sim, double tau)
{
    const std::vector<double>& t = sim->sched_tau;
    const std::vector<double>& v = sim->sched_s;
    if (t.empty()) return sim->p.s;
    if (tau <= t.front()) return v.front();
    for (size_t k = 1; k < t.size(); ++k)
        if (tau <= t[k]) return v[k - 1] + (tau - t[k - 1]) / (t[k] - t[k - 1]) * (v[k] - v[k - 1]);
    return v.back();
}
double e_of(const ahs_sim* sim, double a, double tau) { return sim->p.e * std::pow(a, s_of(sim, tau) - 1.0); }
double lambda_of(const ahs_sim* sim, double a, double tau) { return sim->p.lambda * std::pow(a, 2.0 * (s_of(sim, tau) - 1.0)); }

// Coefficients of Eqs. 4-5 for the step n -> n+1 (L55-57): scale factors at tau_n -+ dt/2 and tau_n.
StepCoef step_coefficients(const ahs_sim* sim, int64_t n)
{
    const ahs_params& p = sim->p;
    const double tau = tau_of(p, n);
    const double a_m = scale_factor(p, tau - 0.5 * p.dt), a_0 = scale_factor(p, tau), a_p = scale_factor(p, tau + 0.5 * p.dt);
    const double e_m = e_of(sim, a_m, tau - 0.5 * p.dt), e_0 = e_of(sim, a_0, tau), e_p = e_of(sim, a_p, tau + 0.5 * p.dt);   // each at its own level
    StepCoef c;
    const double r_mp = a_m / a_p, r_0p = a_0 / a_p, q_0p = a_0 * a_0 / a_p;
    c.c1 = r_mp * r_mp;                                       // (a_{n-1/2}/a_{n+1/2})^2
    c.c2 = p.dt / (p.dx * p.dx) * r_0p * r_0p;                // dt/dx^2 (a_n/a_{n+1/2})^2
    c.c3 = p.dt * q_0p * q_0p * lambda_of(sim, a_0, tau) * 0.5;   // dt (a_n^2/a_{n+1/2})^2 lambda_n/2
    c.d1 = (e_p / e_m) * (e_p / e_m);                         // (e_{n+1/2}/e_{n-1/2})^2
    c.d2 = 2.0 * p.dt * a_0 * a_0 * e_p * e_p;                // 2 dt a_n^2 e_{n+1/2}^2
    c.d3 = p.dt / (p.dx * p.dx) * (e_p / e_0) * (e_p / e_0);  // dt/dx^2 (e_{n+1/2}/e_n)^2
    c.dt = p.dt;
    c.sigma2 = p.sigma * p.sigma;
    return c;
}

DiagCoef diag_coefficients(const ahs_sim* sim, int64_t n)
{
    const ahs_params& p = sim->p;
    const double tau = tau_of(p, n);
    const double a = scale_factor(p, tau), a_h = scale_factor(p, tau - 0.5 * p.dt);
    const double ea = e_of(sim, a, tau), e_h = e_of(sim, a_h, tau - 0.5 * p.dt);
    DiagCoef c;
    c.inv_dx2 = 1.0 / (p.dx * p.dx);
    c.gauge_norm = 1.0 / (2.0 * ea * ea * a * a * p.dx * p.dx);
    c.cB = p.c_B != 0.0 ? p.c_B : 1.0;
    c.cE = p.c_E != 0.0 ? p.c_E : 1.0;
    c.pot_coef = 0.25 * a * a * lambda_of(sim, a, tau);
    c.sigma2 = p.sigma * p.sigma;
    c.gauss_rhs = 2.0 * p.dx * p.dx * e_h * e_h * a_h * a_h;   // = 2 dx^2 e0^2 a_h^(2s) for a constant s
    return c;
}

template <typename T>
int do_step(ahs_sim* s)
{
    FieldPtrs<T> f;
    const int in = s->cur ? PHI_RE1 : PHI_RE0, out = s->cur ? PHI_RE0 : PHI_RE1;
    f.phi_re = slot<T>(s, in); f.phi_im = slot<T>(s, in + 1);
    f.phi_re_out = slot<T>(s, out); f.phi_im_out = slot<T>(s, out + 1);
    for (int i = 0; i < 3; ++i) {
        f.th[i] = slot<T>(s, in + 2 + i);
        f.th_out[i] = slot<T>(s, out + 2 + i);
        f.eps[i] = slot<T>(s, EPS0 + i);
    }
    f.pi_re = slot<T>(s, PI_RE); f.pi_im = slot<T>(s, PI_IM);
    const StepCoef c = step_coefficients(s, s->step);
    GhostPtrs<T> gh;
    const int ob = s->cur ^ 1;
    for (int i = 0; i < 5; ++i) { gh.lo[i] = (T*)s->ghost_lo[ob][i]; gh.hi[i] = (T*)s->ghost_hi[ob][i]; }
    gh.eps2_hi = (T*)s->ghost_eps2_hi;
    return s->kernel == AHS_KERNEL_MARCH ? launch_step_march<T>(f, s->p.N, s->zr, &gh, c, s->step_maps_ok ? &s->step_maps[s->cur] : nullptr, s->opt, s->stream)
                                         : launch_step_generic<T>(f, s->p.N, c, s->stream);
}

template <typename T>
int do_diag(ahs_sim* s)
{
    DiagPtrs<T> f;
    const int in = s->cur ? PHI_RE1 : PHI_RE0;
    f.phi_re = slot<T>(s, in); f.phi_im = slot<T>(s, in + 1);
    for (int i = 0; i < 3; ++i) { f.th[i] = slot<T>(s, in + 2 + i); f.eps[i] = slot<T>(s, EPS0 + i); }
    f.pi_re = slot<T>(s, PI_RE); f.pi_im = slot<T>(s, PI_IM);
    const DiagCoef c = diag_coefficients(s, s->step);
    return s->kernel == AHS_KERNEL_MARCH
               ? launch_diag_march<T>(f, s->p.N, s->zr, c, s->partials, kMaxDiagPartials, s->result,
                                      // the doubt list: the shadow buffer, from its first OWN plane on (a slab's ghost planes there
                                      // belong to the neighbours' next step)
                                      slot<T>(s, s->cur ? PHI_RE0 : PHI_RE1) + (size_t)s->zr.zbase * s->p.N * s->p.N,
                                      5 * s->array_bytes - (size_t)s->zr.zbase * s->p.N * s->p.N * sizeof(T),
                                      s->diag_map_ok ? &s->diag_map[s->cur] : nullptr, s->opt, s->stream)   // shadow buffer: dead between steps
               : launch_diag_generic<T>(f, s->p.N, c, s->partials, kMaxDiagPartials, s->result, s->stream);
}

// The record of a diagnostics pass (raw sums of the reduction) -> the quantities of include/ahs.h
void fill_diag(ahs_diag* out, const ahs_params& p, int64_t diag_step, double nsites, const DiagPartial& r)
{
    std::memset(out, 0, sizeof(*out));
    out->step = diag_step;
    out->tau = tau_of(p, diag_step);
    out->n_pierced = r.n_pierced;
    out->sum_abs_w = r.sum_abs_w;
    out->L = (M_PI / 6.0) * p.dx * (double)r.n_pierced;                     // L93
    const double box = (double)p.N * p.dx;
    out->xi = r.n_pierced ? std::sqrt(box * box * box / out->L) : INFINITY; // L88
    out->v2_num = r.num;
    out->v2_den = r.den;
    const double R = r.num / r.den;                                          // Eq. 10
    out->v2 = 2.0 * R / (1.0 + R);                                           // Eq. 9
    out->mean_lagrangian = r.lsum / nsites;
    out->gauss_max = r.gmax;
    out->gauss_rhs_rms = std::sqrt(r.rhs2 / nsites);
    out->nonfinite = r.nonfinite ? 1 : 0;
    out->v2v_num = r.vnum;
    out->v2v_den = r.vden;
    const double Rv = r.vnum / r.vden;
    out->v2_V = 2.0 * Rv / (1.0 + Rv);
    out->xi_L = std::sqrt(-(2.0 * M_PI * p.sigma * p.sigma) / out->mean_lagrangian);   // mu = 2 pi sigma^2 (R20)
    out->eos_num = r.wnum;
    out->eos_den = r.wden;
    out->v2_omega = 0.5 * (1.0 + 3.0 * r.wnum / r.wden);                                 // Eq. 12
}

int check_sim(const ahs_sim* s)
{
    if (!s) return fail(AHS_ERR_INVALID_ARG, "null handle");
    return AHS_OK;
}

// Every entry point runs on the handle's device whatever the caller's current device is, and puts the caller's device
// back on return: one host thread may drive handles on several GPUs (replicas).
class DeviceGuard {
public:
    explicit DeviceGuard(int device) : prev_(-1), ok_(true)
    {
        int cur = -1;
        if (cudaGetDevice(&cur) != cudaSuccess) { ok_ = false; return; }
        if (cur != device) {
            if (cudaSetDevice(device) != cudaSuccess) { ok_ = false; return; }
            prev_ = cur;
        }
    }
    ~DeviceGuard() { if (prev_ >= 0) cudaSetDevice(prev_); }
    bool ok() const { return ok_; }
private:
    int prev_;
    bool ok_;
};

#define AHS_ENTER(s)                                                                                         \
    if (int r_ = check_sim(s)) return r_;                                                                    \
    DeviceGuard guard_((s)->device);                                                                         \
    if (!guard_.ok()) return fail(AHS_ERR_CUDA, "cannot make device %d current: %s", (s)->device, cudaGetErrorString(cudaGetLastError()))

}  // namespace

extern "C" {

const char* ahs_last_error(void) { return g_err; }
const char* ahs_version(void) { return "ahs 0.1 sm_100a"; }

size_t ahs_required_bytes(int32_t N, int32_t precision)
{
    if (!valid_N(N) || (precision != AHS_F32 && precision != AHS_F64)) return 0;
    const size_t elem = precision == AHS_F32 ? 4 : 8;
    const size_t nsites = (size_t)N * N * N;
    return (size_t)NUM_SLOTS * round256(nsites * elem) + scratch_bytes();
}

ahs_sim* create_sim(const ahs_params* params, const SlabSpec* slab)
{
    g_err[0] = 0;
    if (!params) { fail(AHS_ERR_INVALID_ARG, "params is NULL"); return nullptr; }
    const ahs_params& p = *params;
    if (!valid_N(p.N)) { fail(AHS_ERR_INVALID_ARG, "N = %d out of range [4, 2048]", p.N); return nullptr; }
    if (p.precision != AHS_F32 && p.precision != AHS_F64) { fail(AHS_ERR_INVALID_ARG, "precision must be AHS_F32 or AHS_F64"); return nullptr; }
    if (p.ic_kind < AHS_IC_RANDOM_PHASE || p.ic_kind > AHS_IC_NONE) { fail(AHS_ERR_INVALID_ARG, "unknown ic_kind %d", p.ic_kind); return nullptr; }
    if (!(p.dx > 0) || !(p.dt > 0) || !(p.lambda > 0) || !(p.e > 0) || !(p.sigma > 0)) {
        fail(AHS_ERR_INVALID_ARG, "dx, dt, lambda, e, sigma must be > 0"); return nullptr;
    }
    if (!std::isfinite(p.m) || !std::isfinite(p.s) || !std::isfinite(p.tau0) || !std::isfinite(p.tau_ref) || p.tau_ref < 0) {
        fail(AHS_ERR_INVALID_ARG, "m, s, tau0 must be finite and tau_ref >= 0"); return nullptr;
    }
    if (p.m != 0.0 && !(p.tau0 - 0.5 * p.dt > 0)) { fail(AHS_ERR_INVALID_ARG, "tau0 - dt/2 must be > 0 when m != 0"); return nullptr; }
    if (!std::isfinite(p.c_B) || p.c_B < 0) { fail(AHS_ERR_INVALID_ARG, "c_B must be finite and >= 0 (0 = default 1)"); return nullptr; }
    if (!std::isfinite(p.c_E) || p.c_E < 0) { fail(AHS_ERR_INVALID_ARG, "c_E must be finite and >= 0 (0 = default 1)"); return nullptr; }
    if (p.kernel < AHS_KERNEL_AUTO || p.kernel > AHS_KERNEL_MARCH) { fail(AHS_ERR_INVALID_ARG, "unknown kernel %d", p.kernel); return nullptr; }
    const bool march_ok = p.precision == AHS_F32 ? march_supported<float>(p.N) : march_supported<double>(p.N);
    if (p.kernel == AHS_KERNEL_MARCH && !march_ok) {
        fail(AHS_ERR_INVALID_ARG, "the z-marching kernel needs N %% %d == 0 (N = %d)", p.precision == AHS_F32 ? 128 : 64, p.N);
        return nullptr;
    }

    int dev = 0;
    cudaError_t ce = cudaGetDevice(&dev);
    if (ce != cudaSuccess) { fail(AHS_ERR_CUDA, "no CUDA device: %s (libahs has no CPU fallback)", cudaGetErrorString(ce)); return nullptr; }

    ahs_sim* s = new (std::nothrow) ahs_sim();
    if (!s) { fail(AHS_ERR_OOM, "host allocation failed"); return nullptr; }
    s->p = p;
    s->nsites = (int64_t)p.N * p.N * p.N;
    s->elem = p.precision == AHS_F32 ? 4 : 8;
    s->zr = slab ? ZRange{ slab->nz, 1, 0, slab->nz + 2 } : ZRange{ p.N, 0, 1, p.N };
    s->z_offset = slab ? slab->z_offset : 0;
    s->nsites_alloc = (int64_t)p.N * p.N * s->zr.nz_alloc;
    s->array_bytes = round256((size_t)s->nsites_alloc * s->elem);
    s->stream = (cudaStream_t)p.stream;
    s->owns_stream = false;
    std::memset(s->ghost_lo, 0, sizeof(s->ghost_lo));
    std::memset(s->ghost_hi, 0, sizeof(s->ghost_hi));
    s->ghost_eps2_hi = nullptr;
    s->copy_lo = s->copy_hi = false;
    std::memset(s->copy_lo_dst, 0, sizeof(s->copy_lo_dst));
    std::memset(s->copy_hi_dst, 0, sizeof(s->copy_hi_dst));
    s->copy_eps2_dst = nullptr;
    s->lo_device = s->hi_device = -1;
    if (slab) {
        if (!march_ok || p.device_buffer) { fail(AHS_ERR_INVALID_ARG, "a z-slab needs the z-marching kernels (N %% %d == 0) and library-owned memory", p.precision == AHS_F32 ? 128 : 64); delete s; return nullptr; }
        if (cudaStreamCreateWithFlags(&s->stream, cudaStreamNonBlocking) != cudaSuccess) { fail(AHS_ERR_CUDA, "cudaStreamCreate: %s", cudaGetErrorString(cudaGetLastError())); delete s; return nullptr; }
        s->owns_stream = true;
    }
    s->cur = 0; s->step = 0; s->launches = 0; s->diag_step = -1; s->device = dev;
    s->kernel = (p.kernel == AHS_KERNEL_AUTO) ? (march_ok ? AHS_KERNEL_MARCH : AHS_KERNEL_GENERIC) : p.kernel;
    s->result_host = nullptr;
    s->opt = MarchOptions{ AHS_STAGING_TENSOR, 0, 0, AHS_TRIG_HARDWARE, 0 };

    const size_t need = (size_t)NUM_SLOTS * s->array_bytes + scratch_bytes();
    if (p.device_buffer) {
        if (p.device_buffer_bytes < need || ((uintptr_t)p.device_buffer & 255)) {
            fail(AHS_ERR_INVALID_ARG, "device_buffer must hold %zu bytes and be 256-byte aligned", need);
            delete s; return nullptr;
        }
        cudaPointerAttributes pa;
        if (cudaPointerGetAttributes(&pa, p.device_buffer) != cudaSuccess || pa.type != cudaMemoryTypeDevice || pa.device != dev) {
            cudaGetLastError();
            fail(AHS_ERR_INVALID_ARG, "device_buffer is not device memory of the current device (%d)", dev);
            delete s; return nullptr;
        }
        s->base = (char*)p.device_buffer; s->owns_buffer = false;
    } else {
        size_t free_b = 0, total_b = 0;
        ce = cudaMemGetInfo(&free_b, &total_b);
        if (ce != cudaSuccess) { fail(AHS_ERR_CUDA, "cudaMemGetInfo: %s", cudaGetErrorString(ce)); delete s; return nullptr; }
        if (need > free_b) { fail(AHS_ERR_OOM, "need %zu bytes of device memory, %zu free", need, free_b); delete s; return nullptr; }
        void* ptr = nullptr;
        ce = cudaMalloc(&ptr, need);
        if (ce != cudaSuccess) { cudaGetLastError(); fail(AHS_ERR_OOM, "cudaMalloc(%zu): %s", need, cudaGetErrorString(ce)); delete s; return nullptr; }
        s->base = (char*)ptr; s->owns_buffer = true;
    }
    s->partials = reinterpret_cast<DiagPartial*>(s->base + (size_t)NUM_SLOTS * s->array_bytes);
    s->result = s->partials + kMaxDiagPartials;
    ce = cudaMallocHost((void**)&s->result_host, sizeof(DiagPartial));
    if (ce != cudaSuccess) { fail(AHS_ERR_CUDA, "cudaMallocHost: %s", cudaGetErrorString(ce)); ahs_destroy(s); return nullptr; }

    s->diag_map_ok = false;
    s->step_maps_ok = false;
    if (s->kernel == AHS_KERNEL_MARCH) {
        s->step_maps_ok = p.precision == AHS_F32
            ? make_step_march_maps<float>(&s->step_maps[0], slot<float>(s, PHI_RE0), p.N, s->zr.nz_alloc, s->array_bytes) &&
              make_step_march_maps<float>(&s->step_maps[1], slot<float>(s, PHI_RE1), p.N, s->zr.nz_alloc, s->array_bytes)
            : make_step_march_maps<double>(&s->step_maps[0], slot<double>(s, PHI_RE0), p.N, s->zr.nz_alloc, s->array_bytes) &&
              make_step_march_maps<double>(&s->step_maps[1], slot<double>(s, PHI_RE1), p.N, s->zr.nz_alloc, s->array_bytes);
        s->diag_map_ok = p.precision == AHS_F32
            ? make_diag_march_map<float>(&s->diag_map[0], slot<float>(s, PHI_RE0), slot<float>(s, EPS0 + 1), p.N, s->zr.nz_alloc, s->array_bytes) &&
              make_diag_march_map<float>(&s->diag_map[1], slot<float>(s, PHI_RE1), slot<float>(s, EPS0 + 1), p.N, s->zr.nz_alloc, s->array_bytes)
            : make_diag_march_map<double>(&s->diag_map[0], slot<double>(s, PHI_RE0), slot<double>(s, EPS0 + 1), p.N, s->zr.nz_alloc, s->array_bytes) &&
              make_diag_march_map<double>(&s->diag_map[1], slot<double>(s, PHI_RE1), slot<double>(s, EPS0 + 1), p.N, s->zr.nz_alloc, s->array_bytes);
    }

    // initial condition (L72): everything zero, then phi from Philox
    ce = cudaMemsetAsync(s->base, 0, (size_t)NUM_SLOTS * s->array_bytes, s->stream);
    if (ce != cudaSuccess) { fail(AHS_ERR_CUDA, "cudaMemsetAsync: %s", cudaGetErrorString(ce)); ahs_destroy(s); return nullptr; }
    if (p.ic_kind != AHS_IC_NONE) {
        const int r = p.precision == AHS_F32
                          ? launch_ic<float>(slot<float>(s, PHI_RE0), slot<float>(s, PHI_IM0), p.N, s->zr.nz_alloc, s->z_offset - s->zr.zbase, p.sigma, p.seed, p.ic_kind, s->stream)
                          : launch_ic<double>(slot<double>(s, PHI_RE0), slot<double>(s, PHI_IM0), p.N, s->zr.nz_alloc, s->z_offset - s->zr.zbase, p.sigma, p.seed, p.ic_kind, s->stream);
        if (r < 0) { fail(AHS_ERR_CUDA, "IC kernel launch: %s", cudaGetErrorString(cudaGetLastError())); ahs_destroy(s); return nullptr; }
        s->launches += r;
    }
    return s;
}

ahs_sim* ahs_create_ex(const ahs_params* params) { return create_sim(params, nullptr); }

ahs_sim* ahs_create(int32_t N, double dx, double dt, double lambda, double e, double sigma, double m, double s, double tau0, uint64_t seed)
{
    ahs_params p;
    std::memset(&p, 0, sizeof(p));
    p.N = N; p.precision = AHS_F32; p.ic_kind = AHS_IC_RANDOM_PHASE; p.kernel = AHS_KERNEL_AUTO;
    p.dx = dx; p.dt = dt; p.lambda = lambda; p.e = e; p.sigma = sigma; p.m = m; p.s = s; p.tau0 = tau0; p.tau_ref = 0.0;
    p.seed = seed;
    return ahs_create_ex(&p);
}

int32_t ahs_step(ahs_sim* s, int32_t n)
{
    AHS_ENTER(s);
    if (!s->zr.periodic) return fail(AHS_ERR_STATE, "a z-slab is stepped through its ahs_group (ahs_group_step keeps the slabs' buffers and ghost planes in step)");
    if (n < 0) return fail(AHS_ERR_INVALID_ARG, "n must be >= 0");
    for (int32_t k = 0; k < n; ++k) {
        const int r = s->p.precision == AHS_F32 ? do_step<float>(s) : do_step<double>(s);
        if (r < 0) return fail(r, "step kernel launch failed at step %lld: %s", (long long)s->step, cudaGetErrorString(cudaGetLastError()));
        s->launches += r;
        s->cur ^= 1;
        s->step += 1;
    }
    return AHS_OK;
}

int32_t ahs_diagnostics_launch(ahs_sim* s)
{
    AHS_ENTER(s);
    if (!s->zr.periodic) return fail(AHS_ERR_STATE, "a z-slab's diagnostics are taken through its ahs_group (ahs_group_diagnostics combines the slabs' sums)");
    const int r = s->p.precision == AHS_F32 ? do_diag<float>(s) : do_diag<double>(s);
    if (r < 0) return fail(r, "diagnostics kernel launch failed: %s", cudaGetErrorString(cudaGetLastError()));
    s->launches += r;
    s->diag_step = s->step;
    return AHS_OK;
}

int32_t ahs_diagnostics_fetch(ahs_sim* s, ahs_diag* out)
{
    AHS_ENTER(s);
    if (!out) return fail(AHS_ERR_INVALID_ARG, "out is NULL");
    if (!s->zr.periodic) return fail(AHS_ERR_STATE, "a z-slab's diagnostics are taken through its ahs_group (ahs_group_diagnostics combines the slabs' sums)");
    if (s->diag_step < 0) return fail(AHS_ERR_STATE, "no diagnostics launch is pending");
    AHS_CUDA(cudaMemcpyAsync(s->result_host, s->result, sizeof(DiagPartial), cudaMemcpyDeviceToHost, s->stream));
    AHS_CUDA(cudaStreamSynchronize(s->stream));
    const DiagPartial& r = *s->result_host;
    fill_diag(out, s->p, s->diag_step, (double)s->nsites, r);
    s->diag_step = -1;
    if (out->nonfinite) return fail(AHS_ERR_NONFINITE, "the lattice holds non-finite field values at step %lld (%llu sites or thread-planes flagged)",
                                    (long long)out->step, (unsigned long long)r.nonfinite);
    return AHS_OK;
}

int32_t ahs_diagnostics_ex(ahs_sim* s, ahs_diag* out)
{
    if (!out) return fail(AHS_ERR_INVALID_ARG, "out is NULL");
    if (int r = ahs_diagnostics_launch(s)) return r;
    return ahs_diagnostics_fetch(s, out);
}

int32_t ahs_diagnostics(ahs_sim* s, double* L, double* v2, double* gauss)
{
    ahs_diag d;
    const int r = ahs_diagnostics_ex(s, &d);
    if (r != AHS_OK && r != AHS_ERR_NONFINITE) return r;
    if (L) *L = d.L;
    if (v2) *v2 = d.v2;
    if (gauss) *gauss = d.gauss_max;
    return r;
}

int32_t ahs_get_fields_native(ahs_sim* s, void* host10)
{
    AHS_ENTER(s);
    if (!s->zr.periodic) return fail(AHS_ERR_STATE, "a z-slab's fields are read and written through its ahs_group");
    if (!host10) return fail(AHS_ERR_INVALID_ARG, "host10 is NULL");
    const size_t bytes = (size_t)s->nsites * s->elem;
    for (int k = 0; k < 10; ++k)
        AHS_CUDA(cudaMemcpyAsync((char*)host10 + (size_t)k * bytes, s->base + (size_t)live_slot(s, k) * s->array_bytes, bytes,
                                 cudaMemcpyDeviceToHost, s->stream));
    AHS_CUDA(cudaStreamSynchronize(s->stream));
    return AHS_OK;
}

int32_t ahs_set_fields_native_async(ahs_sim* s, const void* host10, int64_t step)
{
    AHS_ENTER(s);
    if (!s->zr.periodic) return fail(AHS_ERR_STATE, "a z-slab's fields are read and written through its ahs_group");
    if (!host10) return fail(AHS_ERR_INVALID_ARG, "host10 is NULL");
    if (step < 0) return fail(AHS_ERR_INVALID_ARG, "step must be >= 0");
    const size_t bytes = (size_t)s->nsites * s->elem;
    for (int k = 0; k < 10; ++k)
        AHS_CUDA(cudaMemcpyAsync(s->base + (size_t)live_slot(s, k) * s->array_bytes, (const char*)host10 + (size_t)k * bytes, bytes,
                                 cudaMemcpyHostToDevice, s->stream));
    s->step = step;
    return AHS_OK;
}

int32_t ahs_set_fields_native(ahs_sim* s, const void* host10, int64_t step)
{
    if (int r = ahs_set_fields_native_async(s, host10, step)) return r;
    AHS_ENTER(s);
    AHS_CUDA(cudaStreamSynchronize(s->stream));
    return AHS_OK;
}

// fp64 host interface: for AHS_F64 a straight copy; for AHS_F32 each field is converted on the device through
// the (currently dead) shadow buffer of phi/theta, two arrays of which hold one N^3 array of doubles.
int32_t ahs_get_fields(ahs_sim* s, double* host10)
{
    AHS_ENTER(s);
    if (!host10) return fail(AHS_ERR_INVALID_ARG, "host10 is NULL");
    if (s->p.precision == AHS_F64) return ahs_get_fields_native(s, host10);
    if (!s->zr.periodic) return fail(AHS_ERR_STATE, "a z-slab's fields are read and written through its ahs_group");
    const int shadow = s->cur ? PHI_RE0 : PHI_RE1;   // 5 dead float arrays = room for 2 double arrays
    double* stage = reinterpret_cast<double*>(s->base + (size_t)shadow * s->array_bytes);
    const size_t bytes = (size_t)s->nsites * sizeof(double);
    for (int k = 0; k < 10; ++k) {
        const int r = launch_convert_to_double<float>(slot<float>(s, live_slot(s, k)), stage, s->nsites, s->stream);
        if (r < 0) return fail(AHS_ERR_CUDA, "convert kernel: %s", cudaGetErrorString(cudaGetLastError()));
        s->launches += r;
        AHS_CUDA(cudaMemcpyAsync(host10 + (size_t)k * s->nsites, stage, bytes, cudaMemcpyDeviceToHost, s->stream));
    }
    AHS_CUDA(cudaStreamSynchronize(s->stream));
    return AHS_OK;
}

int32_t ahs_set_fields(ahs_sim* s, const double* host10, int64_t step)
{
    AHS_ENTER(s);
    if (!host10) return fail(AHS_ERR_INVALID_ARG, "host10 is NULL");
    if (step < 0) return fail(AHS_ERR_INVALID_ARG, "step must be >= 0");
    if (s->p.precision == AHS_F64) return ahs_set_fields_native(s, host10, step);
    if (!s->zr.periodic) return fail(AHS_ERR_STATE, "a z-slab's fields are read and written through its ahs_group");
    const int shadow = s->cur ? PHI_RE0 : PHI_RE1;
    double* stage = reinterpret_cast<double*>(s->base + (size_t)shadow * s->array_bytes);
    const size_t bytes = (size_t)s->nsites * sizeof(double);
    for (int k = 0; k < 10; ++k) {
        AHS_CUDA(cudaMemcpyAsync(stage, host10 + (size_t)k * s->nsites, bytes, cudaMemcpyHostToDevice, s->stream));
        const int r = launch_convert_from_double<float>(stage, slot<float>(s, live_slot(s, k)), s->nsites, s->stream);
        if (r < 0) return fail(AHS_ERR_CUDA, "convert kernel: %s", cudaGetErrorString(cudaGetLastError()));
        s->launches += r;
    }
    AHS_CUDA(cudaStreamSynchronize(s->stream));
    s->step = step;
    return AHS_OK;
}

int32_t ahs_field_device_ptr(ahs_sim* s, int32_t k, void** dev_ptr)
{
    AHS_ENTER(s);
    if (k < 0 || k > 9 || !dev_ptr) return fail(AHS_ERR_INVALID_ARG, "field index must be 0..9 and dev_ptr non-NULL");
    *dev_ptr = s->base + (size_t)live_slot(s, k) * s->array_bytes;
    return AHS_OK;
}

int32_t ahs_get_state(ahs_sim* s, int64_t* step, double* tau, int64_t* kernel_launches)
{
    AHS_ENTER(s);
    if (step) *step = s->step;
    if (tau) *tau = tau_of(s->p, s->step);
    if (kernel_launches) *kernel_launches = s->launches;
    return AHS_OK;
}

int32_t ahs_kernel_kind(ahs_sim* s)
{
    AHS_ENTER(s);
    return s->kernel;
}

int32_t ahs_coefficients(ahs_sim* s, int64_t n, double* out6)
{
    AHS_ENTER(s);
    if (!out6 || n < 0) return fail(AHS_ERR_INVALID_ARG, "out6 is NULL or n < 0");
    const StepCoef c = step_coefficients(s, n);
    out6[0] = c.c1; out6[1] = c.c2; out6[2] = c.c3; out6[3] = c.d1; out6[4] = c.d2; out6[5] = c.d3;
    return AHS_OK;
}

int32_t ahs_synchronize(ahs_sim* s)
{
    AHS_ENTER(s);
    AHS_CUDA(cudaStreamSynchronize(s->stream));
    return AHS_OK;
}

int32_t ahs_set_option(ahs_sim* s, int32_t option, int32_t value)
{
    AHS_ENTER(s);
    if (value < 0) return fail(AHS_ERR_INVALID_ARG, "option values are >= 0");
    switch (option) {
        case AHS_OPT_STAGING:
            if (value != AHS_STAGING_TENSOR && value != AHS_STAGING_ROWS) return fail(AHS_ERR_INVALID_ARG, "AHS_OPT_STAGING takes AHS_STAGING_TENSOR or AHS_STAGING_ROWS");
            s->opt.staging = value;
            return AHS_OK;
        case AHS_OPT_STEP_CHUNKS:
        case AHS_OPT_DIAG_CHUNKS:
            if (value > s->zr.nz) return fail(AHS_ERR_INVALID_ARG, "at most %d z-chunks per tile (the z-planes this handle owns)", s->zr.nz);
            (option == AHS_OPT_STEP_CHUNKS ? s->opt.step_chunks : s->opt.diag_chunks) = value;
            return AHS_OK;
        case AHS_OPT_DIAG_TRIG:
            if (value != AHS_TRIG_HARDWARE && value != AHS_TRIG_POLYNOMIAL) return fail(AHS_ERR_INVALID_ARG, "AHS_OPT_DIAG_TRIG takes AHS_TRIG_HARDWARE or AHS_TRIG_POLYNOMIAL");
            s->opt.diag_trig = value;
            return AHS_OK;
        case AHS_OPT_STEP_PDL:
            if (value > 1) return fail(AHS_ERR_INVALID_ARG, "AHS_OPT_STEP_PDL takes 0 or 1");
            s->opt.step_pdl = value;
            return AHS_OK;
        default:
            return fail(AHS_ERR_INVALID_ARG, "unknown option %d", option);
    }
}

int32_t ahs_set_s_schedule(ahs_sim* s, int32_t nknots, const double* tau, const double* s_values)
{
    AHS_ENTER(s);
    if (nknots < 0 || nknots > 4096 || (nknots > 0 && (!tau || !s_values))) return fail(AHS_ERR_INVALID_ARG, "nknots must be 0..4096 with non-NULL arrays");
    for (int32_t k = 0; k < nknots; ++k) {
        if (!std::isfinite(tau[k]) || !std::isfinite(s_values[k])) return fail(AHS_ERR_INVALID_ARG, "knots must be finite");
        if (k > 0 && !(tau[k] > tau[k - 1])) return fail(AHS_ERR_INVALID_ARG, "knot times must increase strictly");
    }
    s->sched_tau.assign(tau, tau + nknots);
    s->sched_s.assign(s_values, s_values + nknots);
    return AHS_OK;
}

int32_t ahs_destroy(ahs_sim* s)
{
    if (!s) return AHS_OK;
    DeviceGuard guard_(s->device);
    cudaStreamSynchronize(s->stream);
    if (s->result_host) cudaFreeHost(s->result_host);
    if (s->owns_buffer && s->base) cudaFree(s->base);
    if (s->owns_stream) cudaStreamDestroy(s->stream);
    delete s;
    return AHS_OK;
}


// ---------------------------------------------------------------------------------------------------------------------------
// ahs_group: one lattice cut into z-slabs, one slab per handle, handles on one or several GPUs of this process (
// the paper's stated next step).  The exchange is part of the step kernel: it stores the new (phi, theta) of
// its boundary planes into the neighbouring slabs' ghost planes (peer memory over NVLink when they live on another GPU), and
// CUDA events order step n+1 of a slab behind step n of its two neighbours.  Nothing spins on the device.
// ---------------------------------------------------------------------------------------------------------------------------
struct ahs_group {
    ahs_params p;
    int P;
    std::vector<ahs_sim*> slab;
    std::vector<cudaEvent_t> done[2];   // done[k][r]: slab r has finished its most recent step of parity k (or later work)
    int parity;                         // parity of the NEXT step's events
    bool have_prev;
    int64_t step;
    std::vector<char> no_peer_lo, no_peer_hi;   // slab r cannot reach the GPU of the slab below / above: that face always goes by copies
    bool poisoned;                      // a step failed after some slabs had already run it: fields inconsistent until they are set again
};

namespace {

// THE slab rules (ahs_slab_layout exports them; slabs.py and the multi-process host tests read them from there): slab r of P owns the
// global planes [r N/P, (r+1) N/P) at its local planes 1 .. N/P, between a ghost plane below (local 0: the top own plane of slab r-1,
// periodically) and above (local N/P + 1: the bottom own plane of slab r+1).
struct SlabLayout { int z_offset, nz, lo, hi, nz_alloc; };
bool slab_layout(int N, int P, int r, SlabLayout* out)
{
    if (!valid_N(N) || P < 1 || P > 64 || N % P != 0 || r < 0 || r >= P) return false;
    const int nz = N / P;
    *out = SlabLayout{ r * nz, nz, (r + P - 1) % P, (r + 1) % P, nz + 2 };
    return true;
}
void wire_faces(ahs_group* g, bool copies);   // defined with the step, below
int lo_of(const ahs_group* g, int r) { SlabLayout l{}; slab_layout(g->p.N, g->P, r, &l); return l.lo; }
int hi_of(const ahs_group* g, int r) { SlabLayout l{}; slab_layout(g->p.N, g->P, r, &l); return l.hi; }

char* plane_ptr(const ahs_sim* s, int slot_index, int local_plane)
{
    return s->base + (size_t)slot_index * s->array_bytes + (size_t)local_plane * s->p.N * s->p.N * s->elem;
}

// slab r's next launch runs behind everything its two neighbours had enqueued when they last recorded done[] -- their last step, or the
// diagnostics pass after it (ahs_group_diagnostics records the event again behind its kernels).  cudaStreamWaitEvent covers only work
// enqueued BEFORE that cudaEventRecord: whatever touches a slab's arrays or ghost planes later must record the event again.
int wait_for_neighbours(ahs_group* g, int r)
{
    if (!g->have_prev) return AHS_OK;
    const int k = g->parity ^ 1;
    for (int nb : { lo_of(g, r), hi_of(g, r) })
        if (nb != r && cudaStreamWaitEvent(g->slab[r]->stream, g->done[k][nb], 0) != cudaSuccess)
            return fail(AHS_ERR_CUDA, "cudaStreamWaitEvent: %s", cudaGetErrorString(cudaGetLastError()));
    return AHS_OK;
}

int group_sync(ahs_group* g)
{
    for (ahs_sim* s : g->slab) {
        DeviceGuard guard(s->device);
        if (cudaStreamSynchronize(s->stream) != cudaSuccess) return fail(AHS_ERR_CUDA, "cudaStreamSynchronize: %s", cudaGetErrorString(cudaGetLastError()));
    }
    return AHS_OK;
}

// ghost planes of the CURRENT (phi, theta) buffer and of eps_2 from the neighbours' boundary planes (after the fields were set from the host)
int refresh_ghosts(ahs_group* g)
{
    if (int r = group_sync(g)) return r;
    for (int r = 0; r < g->P; ++r) {
        ahs_sim* s = g->slab[r];
        const ahs_sim* lo = g->slab[lo_of(g, r)];
        const ahs_sim* hi = g->slab[hi_of(g, r)];
        const size_t plane = (size_t)s->p.N * s->p.N * s->elem;
        DeviceGuard guard(s->device);
        const int b = s->cur ? PHI_RE1 : PHI_RE0;
        for (int i = 0; i < 5; ++i) {
            AHS_CUDA(cudaMemcpyPeerAsync(plane_ptr(s, b + i, 0), s->device, plane_ptr(lo, b + i, lo->zr.nz), lo->device, plane, s->stream));
            AHS_CUDA(cudaMemcpyPeerAsync(plane_ptr(s, b + i, s->zr.nz + 1), s->device, plane_ptr(hi, b + i, 1), hi->device, plane, s->stream));
        }
        AHS_CUDA(cudaMemcpyPeerAsync(plane_ptr(s, EPS2, 0), s->device, plane_ptr(lo, EPS2, lo->zr.nz), lo->device, plane, s->stream));
    }
    return group_sync(g);
}

}  // namespace

int32_t ahs_group_destroy(ahs_group* g)
{
    if (!g) return AHS_OK;
    for (ahs_sim* s : g->slab)
        if (s) { DeviceGuard guard(s->device); cudaStreamSynchronize(s->stream); }
    for (int k = 0; k < 2; ++k)
        for (size_t r = 0; r < g->done[k].size(); ++r)
            if (g->done[k][r]) { DeviceGuard guard(g->slab[r]->device); cudaEventDestroy(g->done[k][r]); }
    for (ahs_sim* s : g->slab) ahs_destroy(s);
    delete g;
    return AHS_OK;
}

ahs_group* ahs_group_create(const ahs_params* params, int32_t nslabs, const int32_t* devices)
{
    g_err[0] = 0;
    if (!params) { fail(AHS_ERR_INVALID_ARG, "params is NULL"); return nullptr; }
    if (nslabs < 1 || nslabs > 64 || !valid_N(params->N) || params->N % nslabs != 0) {
        fail(AHS_ERR_INVALID_ARG, "nslabs must be in 1..64 and divide N"); return nullptr;
    }
    if (params->N / nslabs > 2047) {   // the diagnostics march addresses a slab's planes (ghost plane below included) with 11 bits
        fail(AHS_ERR_INVALID_ARG, "a slab holds at most 2047 z-planes: cut N = %d into at least 2 slabs", params->N); return nullptr;
    }
    if (params->device_buffer || params->stream) { fail(AHS_ERR_INVALID_ARG, "a group owns its memory and streams: device_buffer and stream must be NULL"); return nullptr; }
    int ndev = 0, home = 0;
    if (cudaGetDeviceCount(&ndev) != cudaSuccess || ndev < 1 || cudaGetDevice(&home) != cudaSuccess) {
        cudaGetLastError();
        fail(AHS_ERR_CUDA, "no CUDA device (libahs has no CPU fallback)"); return nullptr;
    }
    ahs_group* g = new (std::nothrow) ahs_group();
    if (!g) { fail(AHS_ERR_OOM, "host allocation failed"); return nullptr; }
    g->p = *params; g->P = nslabs; g->parity = 0; g->have_prev = false; g->step = 0; g->poisoned = false;
    g->slab.assign(nslabs, nullptr);
    g->done[0].assign(nslabs, nullptr); g->done[1].assign(nslabs, nullptr);
    for (int r = 0; r < nslabs; ++r) {
        const int dev = devices ? devices[r] : home;
        if (dev < 0 || dev >= ndev) { fail(AHS_ERR_INVALID_ARG, "device %d of slab %d does not exist (%d devices)", dev, r, ndev); ahs_group_destroy(g); return nullptr; }
        DeviceGuard guard(dev);
        ahs_params p = *params;
        p.kernel = AHS_KERNEL_MARCH;
        SlabLayout lay{};
        slab_layout(params->N, nslabs, r, &lay);
        SlabSpec spec = { lay.nz, lay.z_offset };
        g->slab[r] = create_sim(&p, &spec);
        if (!g->slab[r]) { ahs_group_destroy(g); return nullptr; }
        for (int k = 0; k < 2; ++k)
            if (cudaEventCreateWithFlags(&g->done[k][r], cudaEventDisableTiming) != cudaSuccess) {
                fail(AHS_ERR_CUDA, "cudaEventCreate: %s", cudaGetErrorString(cudaGetLastError())); ahs_group_destroy(g); return nullptr;
            }
    }
    // peer access between neighbouring slabs on different devices (a pair without it exchanges by copies), then every slab's targets
    g->no_peer_lo.assign(nslabs, 0); g->no_peer_hi.assign(nslabs, 0);
    for (int r = 0; r < nslabs; ++r)
        for (int side = 0; side < 2; ++side) {
            const int nb = side ? hi_of(g, r) : lo_of(g, r);
            const int a = g->slab[r]->device, b = g->slab[nb]->device;
            if (a == b) continue;
            int can = 0;
            DeviceGuard guard(a);
            if (cudaDeviceCanAccessPeer(&can, a, b) != cudaSuccess || !can) {
                cudaGetLastError();
                (side ? g->no_peer_hi : g->no_peer_lo)[r] = 1;
                continue;
            }
            const cudaError_t e = cudaDeviceEnablePeerAccess(b, 0);
            if (e != cudaSuccess && e != cudaErrorPeerAccessAlreadyEnabled) { fail(AHS_ERR_CUDA, "cudaDeviceEnablePeerAccess: %s", cudaGetErrorString(e)); ahs_group_destroy(g); return nullptr; }
            cudaGetLastError();
        }
    wire_faces(g, false);
    if (group_sync(g) != AHS_OK) { ahs_group_destroy(g); return nullptr; }
    return g;
}

namespace {

// Where each slab's boundary planes go.  A face takes the step kernel's own stores into the neighbour's ghost planes (peer memory
// when the neighbour lives on another GPU) unless the two GPUs have no peer access or `copies` is set; then the kernel gets no
// pointer for that face and step_slab sends the same planes with cudaMemcpyPeerAsync (which needs no peer access: the driver
// stages through the host if it must).  Same values either way: the fields do not depend on the mode.
void wire_faces(ahs_group* g, bool copies)
{
    for (int r = 0; r < g->P; ++r) {
        ahs_sim* s = g->slab[r];
        const ahs_sim* lo = g->slab[lo_of(g, r)];
        const ahs_sim* hi = g->slab[hi_of(g, r)];
        s->copy_lo = copies || g->no_peer_lo[r];
        s->copy_hi = copies || g->no_peer_hi[r];
        s->lo_device = lo->device;
        s->hi_device = hi->device;
        for (int ob = 0; ob < 2; ++ob) {
            const int b = ob ? PHI_RE1 : PHI_RE0;
            for (int i = 0; i < 5; ++i) {
                void* to_lo = plane_ptr(lo, b + i, lo->zr.nz + 1);   // my bottom plane is the lower neighbour's ghost above
                void* to_hi = plane_ptr(hi, b + i, 0);               // my top plane is the upper neighbour's ghost below
                s->ghost_lo[ob][i] = s->copy_lo ? nullptr : to_lo;
                s->ghost_hi[ob][i] = s->copy_hi ? nullptr : to_hi;
                s->copy_lo_dst[ob][i] = s->copy_lo ? to_lo : nullptr;
                s->copy_hi_dst[ob][i] = s->copy_hi ? to_hi : nullptr;
            }
        }
        void* eps2_to_hi = plane_ptr(hi, EPS2, 0);
        s->ghost_eps2_hi = s->copy_hi ? nullptr : eps2_to_hi;
        s->copy_eps2_dst = s->copy_hi ? eps2_to_hi : nullptr;
    }
}

// the faces that go by copies: the new (phi, theta) of the bottom / top own plane (and eps_2 of the top plane) of the buffer the step
// just wrote, enqueued on the slab's stream behind the step kernel and in front of the event its neighbours wait for
int copy_faces(ahs_sim* s, int out_buffer)
{
    const size_t plane = (size_t)s->p.N * s->p.N * s->elem;
    const int b = out_buffer ? PHI_RE1 : PHI_RE0;
    for (int i = 0; i < 5; ++i) {
        if (s->copy_lo) AHS_CUDA(cudaMemcpyPeerAsync(s->copy_lo_dst[out_buffer][i], s->lo_device, plane_ptr(s, b + i, 1), s->device, plane, s->stream));
        if (s->copy_hi) AHS_CUDA(cudaMemcpyPeerAsync(s->copy_hi_dst[out_buffer][i], s->hi_device, plane_ptr(s, b + i, s->zr.nz), s->device, plane, s->stream));
    }
    if (s->copy_hi) AHS_CUDA(cudaMemcpyPeerAsync(s->copy_eps2_dst, s->hi_device, plane_ptr(s, EPS2, s->zr.nz), s->device, plane, s->stream));
    return AHS_OK;
}

const char kPoisoned[] = "an earlier ahs_group_step failed part-way through a step: the slabs' fields are inconsistent until ahs_group_set_fields_native sets them again";

// one slab's share of one step: wait for the neighbours' last step, launch, record
int step_slab(ahs_group* g, int r)
{
    ahs_sim* s = g->slab[r];
    DeviceGuard guard(s->device);
    if (!guard.ok()) return fail(AHS_ERR_CUDA, "cannot make device %d current", s->device);
    if (int e = wait_for_neighbours(g, r)) return e;
    const int rc = s->p.precision == AHS_F32 ? do_step<float>(s) : do_step<double>(s);
    if (rc < 0) return fail(rc, "step kernel launch failed on slab %d at step %lld: %s", r, (long long)s->step, cudaGetErrorString(cudaGetLastError()));
    s->launches += rc;
    if (s->copy_lo || s->copy_hi)
        if (int e = copy_faces(s, s->cur ^ 1)) return e;
    AHS_CUDA(cudaEventRecord(g->done[g->parity][r], s->stream));
    return AHS_OK;
}

}  // namespace

int32_t ahs_group_step(ahs_group* g, int32_t n)
{
    if (!g) return fail(AHS_ERR_INVALID_ARG, "null group");
    if (g->poisoned) return fail(AHS_ERR_STATE, "%s", kPoisoned);
    if (n < 0) return fail(AHS_ERR_INVALID_ARG, "n must be >= 0");
    for (int32_t k = 0; k < n; ++k) {
        for (int r = 0; r < g->P; ++r)
            if (int e = step_slab(g, r)) {
                // slabs 0..r-1 have kicked their momenta in place and stored into their neighbours' ghost planes, the others have
                // not, and no buffer has been flipped: a retry would step those slabs twice.  Refuse further work on these fields.
                g->poisoned = true;
                return e;
            }
        for (ahs_sim* s : g->slab) { s->cur ^= 1; s->step += 1; }
        g->parity ^= 1;
        g->have_prev = true;
        g->step += 1;
    }
    return AHS_OK;
}

int32_t ahs_group_diagnostics(ahs_group* g, ahs_diag* out)
{
    if (!g || !out) return fail(AHS_ERR_INVALID_ARG, "null group or out");
    if (g->poisoned) return fail(AHS_ERR_STATE, "%s", kPoisoned);
    for (int r = 0; r < g->P; ++r) {
        ahs_sim* s = g->slab[r];
        DeviceGuard guard(s->device);
        if (int e = wait_for_neighbours(g, r)) return e;     // the ghosts it reads are the neighbours' last step
        const int rc = s->p.precision == AHS_F32 ? do_diag<float>(s) : do_diag<double>(s);
        if (rc < 0) return fail(rc, "diagnostics kernel launch failed on slab %d: %s", r, cudaGetErrorString(cudaGetLastError()));
        s->launches += rc;
        AHS_CUDA(cudaMemcpyAsync(s->result_host, s->result, sizeof(DiagPartial), cudaMemcpyDeviceToHost, s->stream));
    }
    // The neighbours' next step stores into this slab's ghost planes, and eps_2's ghost plane -- which this pass's Gauss residual reads
    // -- is single-buffered: that step must run behind this pass.  Record the event the neighbours will wait on again, behind the
    // diagnostics kernels (after every slab's waits above were enqueued, so that the passes themselves do not wait for one another);
    // the ordering then holds without the host synchronise below.
    for (int r = 0; r < g->P; ++r) {
        ahs_sim* s = g->slab[r];
        DeviceGuard guard(s->device);
        AHS_CUDA(cudaEventRecord(g->done[g->parity ^ 1][r], s->stream));
    }
    g->have_prev = true;
    DiagPartial t;
    std::memset(&t, 0, sizeof(t));
    for (int r = 0; r < g->P; ++r) {   // fixed order: the result does not depend on which slab finishes first
        ahs_sim* s = g->slab[r];
        DeviceGuard guard(s->device);
        AHS_CUDA(cudaStreamSynchronize(s->stream));
        const DiagPartial& q = *s->result_host;
        t.n_pierced += q.n_pierced; t.sum_abs_w += q.sum_abs_w; t.num += q.num; t.den += q.den; t.lsum += q.lsum;
        t.gmax = q.gmax > t.gmax || q.gmax != q.gmax ? q.gmax : t.gmax;
        t.rhs2 += q.rhs2; t.nonfinite += q.nonfinite; t.vnum += q.vnum; t.vden += q.vden; t.wnum += q.wnum; t.wden += q.wden;
    }
    fill_diag(out, g->p, g->step, (double)g->p.N * g->p.N * g->p.N, t);
    if (out->nonfinite) return fail(AHS_ERR_NONFINITE, "the lattice holds non-finite field values at step %lld", (long long)out->step);
    return AHS_OK;
}

// the whole lattice, 10 N^3 values of the storage type in the field order of include/ahs.h, gathered from / scattered to the slabs
int32_t ahs_group_get_fields_native(ahs_group* g, void* host10)
{
    if (!g || !host10) return fail(AHS_ERR_INVALID_ARG, "null group or host10");
    if (g->poisoned) return fail(AHS_ERR_STATE, "%s", kPoisoned);
    const size_t field = (size_t)g->p.N * g->p.N * g->p.N * g->slab[0]->elem;
    for (ahs_sim* s : g->slab) {
        DeviceGuard guard(s->device);
        const size_t plane = (size_t)s->p.N * s->p.N * s->elem;
        for (int k = 0; k < 10; ++k)
            AHS_CUDA(cudaMemcpyAsync((char*)host10 + (size_t)k * field + (size_t)s->z_offset * plane, plane_ptr(s, live_slot(s, k), 1),
                                     plane * s->zr.nz, cudaMemcpyDeviceToHost, s->stream));
    }
    return group_sync(g);
}

int32_t ahs_group_set_fields_native(ahs_group* g, const void* host10, int64_t step)
{
    if (!g || !host10 || step < 0) return fail(AHS_ERR_INVALID_ARG, "null group or host10, or step < 0");
    if (int r = group_sync(g)) return r;
    const size_t field = (size_t)g->p.N * g->p.N * g->p.N * g->slab[0]->elem;
    for (ahs_sim* s : g->slab) {
        DeviceGuard guard(s->device);
        const size_t plane = (size_t)s->p.N * s->p.N * s->elem;
        for (int k = 0; k < 10; ++k)
            AHS_CUDA(cudaMemcpyAsync(plane_ptr(s, live_slot(s, k), 1), (const char*)host10 + (size_t)k * field + (size_t)s->z_offset * plane,
                                     plane * s->zr.nz, cudaMemcpyHostToDevice, s->stream));
        s->step = step;
    }
    g->step = step;
    const int rc = refresh_ghosts(g);
    if (rc == AHS_OK) g->poisoned = false;   // every live field, ghost plane and step counter has just been written
    return rc;
}

int32_t ahs_group_synchronize(ahs_group* g)
{
    if (!g) return fail(AHS_ERR_INVALID_ARG, "null group");
    return group_sync(g);
}

int32_t ahs_group_set_exchange(ahs_group* g, int32_t mode)
{
    if (!g) return fail(AHS_ERR_INVALID_ARG, "null group");
    if (mode != AHS_EXCHANGE_STORES && mode != AHS_EXCHANGE_COPIES) return fail(AHS_ERR_INVALID_ARG, "mode must be AHS_EXCHANGE_STORES or AHS_EXCHANGE_COPIES");
    if (int r = group_sync(g)) return r;      // no step in flight while the targets change
    wire_faces(g, mode == AHS_EXCHANGE_COPIES);
    return AHS_OK;
}

int32_t ahs_group_exchange_faces(ahs_group* g, int32_t* copied_faces)
{
    if (!g) return fail(AHS_ERR_INVALID_ARG, "null group");
    int n = 0;
    for (const ahs_sim* s : g->slab) n += (s->copy_lo ? 1 : 0) + (s->copy_hi ? 1 : 0);
    if (copied_faces) *copied_faces = n;
    return AHS_OK;
}

int32_t ahs_slab_layout(int32_t N, int32_t nslabs, int32_t r, int32_t* out5)
{
    SlabLayout l{};
    if (!out5) return fail(AHS_ERR_INVALID_ARG, "out5 is NULL");
    if (!slab_layout(N, nslabs, r, &l)) return fail(AHS_ERR_INVALID_ARG, "nslabs must be in 1..64 and divide N (4..2048), and 0 <= r < nslabs");
    out5[0] = l.z_offset; out5[1] = l.nz; out5[2] = l.lo; out5[3] = l.hi; out5[4] = l.nz_alloc;
    return AHS_OK;
}

int32_t ahs_group_slab_count(ahs_group* g) { return g ? g->P : fail(AHS_ERR_INVALID_ARG, "null group"); }

ahs_sim* ahs_group_slab(ahs_group* g, int32_t r)
{
    if (!g || r < 0 || r >= g->P) { fail(AHS_ERR_INVALID_ARG, "null group or slab index out of range"); return nullptr; }
    return g->slab[r];
}

}  // extern "C"

// ---------------------------------------------------------------------------------------------------------------------------
// ahs_diagnostics_static (include/ahs.h): the diagnostics of a snapshot the CALLER holds, for callers that may not allocate -- a run
// that has filled HBM, a hook inside another framework's step loop, a loop that must stay out of the driver's allocator (cudaMalloc
// and cudaFree also stall every stream of the device).  No handle, no cudaMalloc / cudaMallocHost / cudaFree, no stream or event
// creation: the reduction's per-block records, which a handle keeps behind its field arrays, live in the array below, which is part
// of the library image.  The kernel is the one-thread-per-site diagnostics kernel of AHS_KERNEL_GENERIC handles, unchanged and with
// the same launch shape, given the array's device address instead of a handle's scratch.
// ---------------------------------------------------------------------------------------------------------------------------
static_assert(sizeof(DiagPartial) == 96, "AHS_STATIC_SCRATCH_BYTES in include/ahs.h counts 96-byte records");
static_assert(AHS_STATIC_SCRATCH_BYTES >= sizeof(DiagPartial) * (AHS_STATIC_MAX_RECORDS + 1) && AHS_STATIC_SCRATCH_BYTES % 256 == 0,
              "the array holds AHS_STATIC_MAX_RECORDS block records and the result record");

// AHS_STATIC_MAX_RECORDS block records followed by the result record.  Every GPU this process uses libahs on holds these 444.25 KiB
// from the moment this file's code is loaded onto it until the process exits.  One array per device, shared by every call: it keeps
// the last call's contents, and calls that overlap on the GPU race on it (see the header).
// In HOST code the name g_static_scratch is only the key cudaGetSymbolAddress takes.  It is not a device address: a kernel handed
// `g_static_scratch` (or &g_static_scratch[k]) from the host would be reading and writing host memory, or faulting.  Host code passes
// static_scratch_address()'s result; device code of this file may use the name itself (static_clear_result does).
static __device__ __align__(256) unsigned char g_static_scratch[AHS_STATIC_SCRATCH_BYTES];

namespace {

constexpr int kStaticMaxDevices = 64;
// the array's device address on each device (every device has its own copy at its own address); NULL = not looked up yet
std::atomic<void*> g_static_address[kStaticMaxDevices];

// Set-up, once per device, with that device current (`device` is the caller's current device): the first call asks the runtime for
// the address of this device's copy -- which also makes the driver load this file's code, and the array with it, onto the GPU, so it
// belongs before any stream capture -- later calls read the stored pointer.  Two threads racing on the first call both look the
// address up and store the same value.
int static_scratch_address(int device, DiagPartial** out)
{
    if (device < 0 || device >= kStaticMaxDevices)
        return fail(AHS_ERR_INVALID_ARG, "ahs_diagnostics_static serves device ordinals 0..%d (current device: %d)", kStaticMaxDevices - 1, device);
    void* p = g_static_address[device].load(std::memory_order_acquire);
    if (!p) {
        const cudaError_t e = cudaGetSymbolAddress(&p, g_static_scratch);
        if (e != cudaSuccess || !p) {
            cudaGetLastError();
            return fail(AHS_ERR_CUDA, "cudaGetSymbolAddress(static scratch) on device %d: %s", device, cudaGetErrorString(e));
        }
        g_static_address[device].store(p, std::memory_order_release);
    }
    *out = static_cast<DiagPartial*>(p);
    return AHS_OK;
}

// The result record of the call before must not be readable as this call's: zero it (device code names the array directly).
__global__ void static_clear_result()
{
    unsigned long long* rec = reinterpret_cast<unsigned long long*>(g_static_scratch + sizeof(DiagPartial) * AHS_STATIC_MAX_RECORDS);
    if (threadIdx.x < sizeof(DiagPartial) / sizeof(unsigned long long)) rec[threadIdx.x] = 0ull;
}

// how many block records the one-thread-per-site diagnostics kernel writes for an N^3 lattice (launch_diag_generic's grid)
int64_t static_records_needed(int64_t N)
{
    const int64_t blocks = (N * N * N + 127) / 128;
    return blocks < 148 * 32 ? blocks : 148 * 32;
}

template <typename T>
int static_diag(const ahs_params& p, const void* const* fields10, const DiagCoef& c, DiagPartial* scratch, cudaStream_t st)
{
    DiagPtrs<T> f;
    f.phi_re = (const T*)fields10[0]; f.phi_im = (const T*)fields10[1];
    f.pi_re = (const T*)fields10[2]; f.pi_im = (const T*)fields10[3];
    for (int i = 0; i < 3; ++i) { f.th[i] = (const T*)fields10[4 + i]; f.eps[i] = (const T*)fields10[7 + i]; }
    return launch_diag_generic<T>(f, p.N, c, scratch, AHS_STATIC_MAX_RECORDS, scratch + AHS_STATIC_MAX_RECORDS, st);
}

}  // namespace

extern "C" int32_t ahs_diagnostics_static(const ahs_params* params, const void* const* fields10, int64_t step, ahs_diag* out)
{
    if (!params || !fields10 || !out) return fail(AHS_ERR_INVALID_ARG, "params, fields10 and out must not be NULL");
    const ahs_params& p = *params;
    if (p.N < 4 || p.N > AHS_STATIC_MAX_N)
        return fail(AHS_ERR_INVALID_ARG, "N = %d is outside 4..%d, the lattice sizes ahs_diagnostics_static accepts", p.N, (int)AHS_STATIC_MAX_N);
    const int64_t need = static_records_needed(p.N);
    if (need > AHS_STATIC_MAX_RECORDS)
        return fail(AHS_ERR_INVALID_ARG, "N = %d needs %lld reduction records, the static scratch array holds %d (%d bytes)", p.N,
                    (long long)need, (int)AHS_STATIC_MAX_RECORDS, (int)AHS_STATIC_SCRATCH_BYTES);
    if (p.precision != AHS_F32 && p.precision != AHS_F64) return fail(AHS_ERR_INVALID_ARG, "precision must be AHS_F32 or AHS_F64");
    if (!(p.dx > 0) || !(p.dt > 0) || !(p.lambda > 0) || !(p.e > 0) || !(p.sigma > 0)) return fail(AHS_ERR_INVALID_ARG, "dx, dt, lambda, e, sigma must be > 0");
    if (!std::isfinite(p.m) || !std::isfinite(p.s) || !std::isfinite(p.tau0) || !std::isfinite(p.tau_ref) || p.tau_ref < 0)
        return fail(AHS_ERR_INVALID_ARG, "m, s, tau0 must be finite and tau_ref >= 0");
    if (p.m != 0.0 && !(p.tau0 - 0.5 * p.dt > 0)) return fail(AHS_ERR_INVALID_ARG, "tau0 - dt/2 must be > 0 when m != 0");
    if (!std::isfinite(p.c_B) || p.c_B < 0 || !std::isfinite(p.c_E) || p.c_E < 0) return fail(AHS_ERR_INVALID_ARG, "c_B, c_E must be finite and >= 0 (0 = default 1)");
    if (step < 0) return fail(AHS_ERR_INVALID_ARG, "step must be >= 0");

    int dev = 0;
    cudaError_t ce = cudaGetDevice(&dev);
    if (ce != cudaSuccess) { cudaGetLastError(); return fail(AHS_ERR_CUDA, "no CUDA device: %s (libahs has no CPU fallback)", cudaGetErrorString(ce)); }
    for (int k = 0; k < 10; ++k) {
        if (!fields10[k]) return fail(AHS_ERR_INVALID_ARG, "fields10[%d] is NULL", k);
        cudaPointerAttributes pa;
        if (cudaPointerGetAttributes(&pa, fields10[k]) != cudaSuccess || (pa.type != cudaMemoryTypeDevice && pa.type != cudaMemoryTypeManaged) ||
            (pa.type == cudaMemoryTypeDevice && pa.device != dev)) {
            cudaGetLastError();
            return fail(AHS_ERR_INVALID_ARG, "fields10[%d] is not device memory of the current device (%d)", k, dev);
        }
    }
    DiagPartial* scratch = nullptr;
    if (int r = static_scratch_address(dev, &scratch)) return r;

    ahs_sim shell{};            // carries the parameters to diag_coefficients (host only: no s(tau) schedule, nothing allocated)
    shell.p = p;
    const DiagCoef c = diag_coefficients(&shell, step);
    cudaStream_t st = (cudaStream_t)p.stream;
    static_clear_result<<<1, 32, 0, st>>>();
    AHS_CUDA(cudaGetLastError());
    const int launched = p.precision == AHS_F32 ? static_diag<float>(p, fields10, c, scratch, st) : static_diag<double>(p, fields10, c, scratch, st);
    if (launched < 0) return fail(launched, "diagnostics kernel launch failed: %s", cudaGetErrorString(cudaGetLastError()));
    DiagPartial rec;            // pageable host memory on this frame: the copy is staged by the driver, the synchronise below ends it
    AHS_CUDA(cudaMemcpyAsync(&rec, scratch + AHS_STATIC_MAX_RECORDS, sizeof(rec), cudaMemcpyDeviceToHost, st));
    AHS_CUDA(cudaStreamSynchronize(st));
    fill_diag(out, p, step, (double)p.N * p.N * p.N, rec);
    if (out->nonfinite) return fail(AHS_ERR_NONFINITE, "the snapshot holds non-finite field values at step %lld (%llu sites flagged)",
                                    (long long)step, (unsigned long long)rec.nonfinite);
    return AHS_OK;
}
