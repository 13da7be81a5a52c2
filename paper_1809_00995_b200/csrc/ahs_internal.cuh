// ahs_internal.cuh -- private declarations shared by the translation units of libahs (CUDA, sm_100a).
// Nothing here is shared with oracle/ (test infrastructure): the two paths have no common code.
#pragma once

#include <cuda.h>
#include <cuda_runtime.h>
#include <stdint.h>

#include <atomic>

#include "../../include/ahs.h"

namespace ahs {

// Field slots inside the device buffer.  phi and theta are double-buffered ("cur" = 0/1) so that one
// fused kernel can kick Pi, eps in place and write the drifted phi', theta' without a race
// (Eqs. 4-7 need phi^n, theta^n of the neighbours while phi^{n+1} is being produced).
enum Slot {
    PHI_RE0 = 0, PHI_IM0, TH0_0, TH1_0, TH2_0,   // buffer 0 of (phi, theta)
    PHI_RE1, PHI_IM1, TH0_1, TH1_1, TH2_1,       // buffer 1
    PI_RE, PI_IM, EPS0, EPS1, EPS2,              // single-buffered momenta
    NUM_SLOTS
};

// The six per-step scalars of Eqs. 4-5 (host, fp64) plus constants, passed by value to the kernels.
struct StepCoef {
    double c1, c2, c3, d1, d2, d3;   // Eq. 4: c1 damping, c2 Laplacian, c3 Higgs force; Eq. 5: d1, d2 current, d3 curl
    double dt;                        // Eqs. 6-7
    double sigma2;                    // sigma^2
};

// Constants of the diagnostics pass for the snapshot after n steps.
struct DiagCoef {
    double inv_dx2;        // 1/dx^2
    double gauge_norm;     // 1 / (2 e(a)^2 a^2 dx^2) with a = a(tau_n)     (Eq. 2 prefactor)
    double cB;             // c_B: factor on the magnetic term in the weight, 1 (R2)
    double cE;             // c_E: factor on the electric term in the weight, 1 (R21)
    double pot_coef;       // a^2 lambda(a) / 4
    double sigma2;
    double gauss_rhs;      // 2 dx^2 e0^2 a_h^(2s), a_h = a(tau_n - dt/2)  (R4)
};

// One record per block / final result of the reduction (fixed 12 x 8 bytes).
struct DiagPartial {
    unsigned long long n_pierced;
    unsigned long long sum_abs_w;
    double num, den, lsum;
    double gmax;
    double rhs2;
    unsigned long long nonfinite;
    double vnum, vden;     // potential-weighted sums: sum K Vp, sum G Vp
    double wnum, wden;     // equation of state, Lagrangian weighted: sum p Lag, sum rho Lag (Eq. 12; R22)
};

// Which z-planes of the allocated arrays a handle owns.  A whole lattice: nz = nz_alloc = N, zbase = 0, periodic in z.  A z-slab
// (ahs_group): nz own planes at local indices zbase = 1 .. nz, a ghost plane below (local 0, the lower neighbour's top
// plane) and above (local nz + 1), no wrap: the neighbours keep the ghosts current (peer stores of the step kernel).
struct ZRange {
    int nz;         // own planes
    int zbase;      // local index of the first own plane
    int periodic;   // wrap z inside the array (whole lattice) or not (slab with ghost planes)
    int nz_alloc;   // planes allocated per array
};

// Where the step kernel also stores the new (phi, theta) of its bottom / top own plane: the neighbouring slabs' ghost planes, in
// THEIR output buffer (device pointers to the first element of the plane; peer memory over NVLink when the slab lives on another
// GPU).  eps2_hi: the upper neighbour's ghost-below plane of eps_2 (the Gauss residual needs eps_2^{x-k_2}).  NULL = none.
template <typename T>
struct GhostPtrs {
    T* lo[5];
    T* hi[5];
    T* eps2_hi;
};

template <typename T>
struct FieldPtrs {
    const T* phi_re; const T* phi_im; const T* th[3];   // level n (read only)
    T* phi_re_out; T* phi_im_out; T* th_out[3];         // level n+1 (other buffer)
    T* pi_re; T* pi_im; T* eps[3];                      // in place
};

template <typename T>
struct DiagPtrs {
    const T* phi_re; const T* phi_im; const T* th[3];
    const T* pi_re; const T* pi_im; const T* eps[3];
};

// Tuning of the marching kernels, set per handle through ahs_set_option (include/ahs.h); 0 = the library's choice.
struct MarchOptions {
    int staging;       // AHS_STAGING_TENSOR (tensor-map TMA where a tile allows it) or AHS_STAGING_ROWS (row copies only)
    int step_chunks;   // z-chunks per tile of the step march
    int diag_chunks;   // z-chunks per tile of the diagnostics march
    int diag_trig;     // AHS_TRIG_HARDWARE or AHS_TRIG_POLYNOMIAL: the sines and cosines of the <v^2> sums (fp32 lattices)
    int step_pdl;      // launch the step march with programmatic stream serialization (its prologue overlaps the previous kernel's tail)
};

// cudaFuncAttributeMaxDynamicSharedMemorySize is per device: set it once on every device a kernel is launched on
// (one static instance per kernel instantiation; handles on different GPUs of one process share the kernels).
struct SmemAttribute {
    std::atomic<unsigned long long> done{ 0ull };
    template <typename K> bool ensure(K kernel, size_t bytes)
    {
        int dev = 0;
        if (cudaGetDevice(&dev) != cudaSuccess) return false;
        const unsigned long long bit = dev < 64 ? 1ull << dev : 0ull;
        if (bit && (done.load(std::memory_order_acquire) & bit)) return true;
        if (cudaFuncSetAttribute(kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)bytes) != cudaSuccess) return false;
        done.fetch_or(bit, std::memory_order_release);
        return true;
    }
};

// ---- kernel launchers (each returns the number of kernels it launched, or a negative ahs error) -------------
// IC on nz_alloc planes starting at global plane z_first (periodic): the Philox counter is the site index of the FULL N^3 lattice
template <typename T> int launch_ic(T* phi_re, T* phi_im, int N, int nz_alloc, int z_first, double sigma, uint64_t seed, int kind, cudaStream_t st);
template <typename T> int launch_step_generic(const FieldPtrs<T>& f, int N, const StepCoef& c, cudaStream_t st);
// TMA descriptors of the step march: the four-array stage and theta_2 of one (phi, theta) buffer
struct StepMaps { CUtensorMap stage, th2, wstage, wth2; };   // w*: the V-wide wrapped halo column of x-edge tiles
template <typename T> int launch_step_march(const FieldPtrs<T>& f, int N, const ZRange& zr, const GhostPtrs<T>* ghosts /* may be NULL */, const StepCoef& c,
                                            const StepMaps* maps /* HOST, may be NULL */, const MarchOptions& opt, cudaStream_t st);
template <typename T> bool make_step_march_maps(StepMaps* out, const void* phi_re_base, int N, int nz_alloc, size_t array_bytes);
template <typename T> bool march_supported(int N);
template <typename T> int launch_diag_generic(const DiagPtrs<T>& f, int N, const DiagCoef& c, DiagPartial* partials,
                                              int max_partials, DiagPartial* result, cudaStream_t st);
// TMA descriptors of the diagnostics march: the five-array forward-halo tile, the V-wide wrapped column of right-edge tiles,
// and the rows y0-1 .. y0+TY-1 of eps_1
struct DiagMaps { CUtensorMap tile, wrap, eps1; };
// `list`: DEVICE scratch of >= 4 N^3 / (16 / sizeof(T)) bytes for the winding doubt list (the dead phi', theta' shadow buffer)
template <typename T> int launch_diag_march(const DiagPtrs<T>& f, int N, const ZRange& zr, const DiagCoef& c, DiagPartial* partials,
                                            int max_partials, DiagPartial* result, void* list, size_t list_bytes,
                                            const DiagMaps* tmap /* HOST, may be NULL: row copies only */, const MarchOptions& opt,
                                            cudaStream_t st);
// tensor maps (TMA descriptors) of the five level-n arrays of one (phi, theta) buffer and of eps_1 for the diagnostics march; false if unavailable
template <typename T> bool make_diag_march_map(DiagMaps* out, const void* phi_re_base, const void* eps1_base, int N, int nz_alloc, size_t array_bytes);
int launch_diag_finish(const DiagPartial* partials, int n, DiagPartial* result, cudaStream_t st);
template <typename T> int launch_convert_from_double(const double* src, T* dst, int64_t n, cudaStream_t st);
template <typename T> int launch_convert_to_double(const T* src, double* dst, int64_t n, cudaStream_t st);

static const int kMaxDiagPartials = 1 << 16;

}  // namespace ahs
