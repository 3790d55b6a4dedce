// clt_internal.h -- shared declarations of libclt's host side (clt_api.cu) and kernels (clt_kernels.cu).
// Product code: shares nothing with oracle/.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>
#include <stddef.h>

namespace clt {

// ---------------------------------------------------------------------------------------------
// Internal HBM layout.  A scalar field is [nphi][nZ][pR] doubles, R fastest.
// Node i of a row sits at column LP + i with LP = 14, so that the first interior node (i = 2) of
// every row is 128-byte aligned (pR is a multiple of 16 doubles and every field base is 256-byte
// aligned).  The R/Z boundary layers are part of the array and are never written by the step
// kernels; phi has no ghost planes (the plane index wraps).
constexpr int LP = 14;

struct Layout {
    int nR, nphi, nZ;
    int pR;             // row pitch in doubles
    long long plane;    // nZ * pR
    long long field;    // nphi * plane
    __host__ __device__ long long at(int i, int k, int j) const {
        return (long long)j * plane + (long long)k * pR + (LP + i);
    }
};

// Indices of the axisymmetric tables ([nZ][pR] each, same row layout as a field plane).
enum Table {
    T_RHO0 = 0, T_P0, T_V0R, T_V0P, T_V0Z, T_B0R, T_B0P, T_B0Z,   // U0 (eqs 11-14)
    T_J0R, T_J0P, T_J0Z,                                          // J0 = curl_c B0 (interior; 0 on boundary layers)
    T_GR_RHO0, T_GZ_RHO0, T_GR_P0, T_GZ_P0,                       // d_R, d_Z of rho0, p0
    T_E0R, T_E0P, T_E0Z,                                          // v0 x B0
    T_GR_V0R, T_GZ_V0R, T_GR_V0P, T_GZ_V0P, T_GR_V0Z, T_GZ_V0Z,   // d_R, d_Z of v0
    T_DIVV0,                                                      // div v0
    T_A0R, T_A0P, T_A0Z,                                          // (v0.grad) v0
    T_COUNT
};

struct Phys {
    double gamma, eta, nu, D, kappa;
    double d_i;              // ion inertial length of the Hall term of eq (5); 0 = resistive MHD
    double cR1, cZ1, cP1;    // 1/(12 h)
    double cR2, cZ2, cP2;    // 1/(12 h^2)
    double dR, dZ, dphi, Lphi;
};

// Parameters of one fused RHS (+ RK4 stage combine) launch.
struct RhsArgs {
    Layout L;
    Phys ph;
    const double *in;     // stage state, 8 fields
    const double *J1;     // 3 fields (the Hall variant reads 3 more right behind them: G)
    const double *Un;     // U^n, 8 fields (modes 2, 3, 4; mode 4 updates it in place through `out`)
    double *acc;          // RK4 accumulator, 8 fields (written by mode 2, read by mode 4)
    double *out;          // K (mode 0) | next stage state (modes 1-3) | U^{n+1} (mode 4), 8 fields
    const double *tab;    // T_COUNT tables
    const double *R;      // R_i, i = -LP .. : pointer already offset so that R[i] is node i; padded with valid numbers
    const double *invR;   // 1/R_i, same indexing
    int phi_chunks;       // number of chunks the phi range is split into (gridDim.z)
    int prefetch;         // issue L2 prefetch hints
    const double *spec;   // pseudo-spectral variant: SPEC_COUNT derivative fields (SpecField)
    // stage coefficients { dt, dt/2, dt/3, dt/6 } in device memory: the fixed-dt table of clt_set_dt or the device clock of
    // clt_step_cfl (so a captured CUDA graph of the step does not bake dt in)
    const double *coef;
    // adaptive stepping (clt_step_cfl): non-null = stage 4 folds the SETDT minimum of the new state into *dtmin_bits
    unsigned long long *dtmin_bits;
    double cfl;
    // rows this context is responsible for (a slab's owned rows; default 2 .. nZ-3): the only rows a stage writes, and the
    // rows whose new state enters the SETDT minimum
    int own_k0, own_k1;
    // NEXT-4: neighbouring slabs of the same process.  Rows k0 .. k1 of a stage's output are also stored into rows
    // k + dk of the neighbour's buffer of the same stage (its ghost rows), straight from the epilogue.  out = nullptr: none.
    struct Peer {
        double *out;
        long long plane, field;
        int k0, k1, dk;
    } peer[2];
};

// clocks of a group of contexts that share one adaptive time step (clt_cfl_commit)
constexpr int DT_GROUP_MAX = 64;
struct DtGroup {
    int n;
    double *clock[DT_GROUP_MAX];
    unsigned long long *dtmin_bits[DT_GROUP_MAX];
    const double *diag6[DT_GROUP_MAX];
};

struct CurlArgs {
    Layout L;
    Phys ph;
    const double *B;      // 3 fields (B_R, B_phi, B_Z of the stage state)
    double *J1;           // 3 fields
    double *G;            // 3 fields: Hall field (written by the Hall variant only)
    const double *spec;   // pseudo-spectral variant: derivative fields (uses SP_DB and, with hall, SP_D1 + 1)
    const double *tab;
    const double *R;
    const double *invR;
    int phi_chunks;
};

// NEXT-2: pseudo-spectral phi derivatives.  Scratch layout: SPEC_COUNT fields.
enum SpecField {
    SP_D1 = 0,        // d/dphi of rho1, p1, v1_R, v1_phi, v1_Z (5 fields)
    SP_D2 = 5,        // d2/dphi2 of the same (5 fields)
    SP_DE = 10,       // d/dphi of E1_R, E1_Z
    SP_DB = 12,       // d/dphi of B1_R, B1_Z
    SPEC_COUNT = 14
};
constexpr int SPEC_MAX_NPHI = 256;

// one phi pre-pass: mode 0 = before the curl (B_R, B_Z; p too when hall), 1 = before the fused RHS kernel
// (rho, p, v: first and second derivative; E1_R, E1_Z: first derivative)
struct SpecArgs {
    Layout L;
    Phys ph;
    const double *U;      // stage state, 8 fields
    const double *J1;     // 3 fields (+ G behind them when hall)
    const double *tab;
    double *out;          // SPEC_COUNT fields
    const double *ctab;   // [2][SPEC_MAX_NPHI]: circulant weights c1[m] (antisymmetric in m), c2[m] (symmetric)
    int mode, hall, has_v0;
};

struct DiagArgs {
    Layout L;
    Phys ph;
    const double *U;
    const double *tab;
    const double *R;
    const double *invR;
    const double *cs;     // cos/sin(2 pi j / nphi), [2][nphi]
    double *partial;      // [nblocks][6]
    double cfl;
    const double *spec_c1;   // non-null: pseudo-spectral d/dphi in div_c B, weights c1[0..nphi-1]
    double ihZ;              // 1 / dZ
    int k_first, k_last;     // rows the sums / the SETDT minimum run over (default 2 .. nZ-3; a slab's owned rows)
    int kd_first, kd_last;   // rows of the max |div_c B| (default 4 .. nZ-5)
};

enum { RHS_MODE_K = 0, RHS_MODE_S1 = 1, RHS_MODE_S2 = 2, RHS_MODE_S3 = 3, RHS_MODE_S4 = 4 };

// kernel launchers (clt_kernels.cu); each returns the cudaGetLastError() of its launch.  configure = true: do not
// launch, only opt the kernel in to its dynamic shared-memory size on the current device (configure_kernels)
cudaError_t launch_tables(const Layout &L, const Phys &ph, double *tab, const double *R, const double *invR,
                          cudaStream_t s);
cudaError_t launch_any_nonzero(const double *x, long long n, int *flag, cudaStream_t s);
cudaError_t launch_copy_boundary(const Layout &L, int nfields, const double *src, double *d0, double *d1, double *d2,
                                 int sm_count, cudaStream_t s);
// rows k0s .. k0s+nrows-1 of nfp = fields * planes slices of `src` (layout Ls) -> rows k0d .. of `dst` (layout Ld)
cudaError_t launch_push_rows(const Layout &Ls, const double *src, int k0s, const Layout &Ld, double *dst, int k0d, int nrows,
                             int sm_count, cudaStream_t s);
cudaError_t launch_zero_boundary(const Layout &L, int nfields, double *dst, int sm_count, cudaStream_t s);
// plain-load variants (kernel variant 1: A/B and parity cross-check of the TMA-fed default)
cudaError_t launch_curl(const CurlArgs &a, cudaStream_t s);
cudaError_t launch_rhs(const RhsArgs &a, int mode, bool has_v0, cudaStream_t s, bool configure = false);
// TMA variant: tmU / tmJ / tmV point to CUtensorMap objects (4-D: pR, nZ, nphi, field) with boxes (TR+4, rhs_tile_z()+4, 1, nf)
// that span the field axis.  Moving reference state (has_v0) or pseudo-spectral scheme: tmU over the stage state with nf = 8,
// tmV unused.  Static reference state with finite differences: tmU with nf = 2 (rho, p), tmV with nf = 3 (v at field 2, B at field 5).  tmJ over J1 with nf = 3
// (hall: 6 fields, J1 then G; the kernel adds d_i * G to E1).
// slab: the context is a slab (owned rows set and / or neighbours linked, RhsArgs::own_k0 .. peer)
cudaError_t launch_rhs_tma(const RhsArgs &a, const void *tmU, const void *tmJ, const void *tmV, int mode, bool has_v0, bool hall,
                           bool spec, bool slab, cudaStream_t s, bool configure = false);
// TMA variant of the curl kernel: tmU is a CUtensorMap over the 8 fields of the stage state with box
// (TR+4, curl_tma_tile_z()+4, 1, 1); hall = also write the Hall field G
cudaError_t launch_curl_tma(const CurlArgs &a, const void *tmU, bool hall, bool spec, cudaStream_t s, bool configure = false);
cudaError_t launch_phi_spectral(const SpecArgs &a, cudaStream_t s, bool configure = false);
int curl_tma_tile_z();
int rhs_tile_z();
cudaError_t launch_dt_commit_group(const DtGroup &g, int init, cudaStream_t s);
cudaError_t launch_dt_commit(double *clock, unsigned long long *dtmin_bits, const double *diag6, int init, cudaStream_t s);
cudaError_t launch_diag(const DiagArgs &a, int nblocks, double *result6, cudaStream_t s, const void *tmU = nullptr, bool configure = false);
int diag_tma_tile_z();
int diag_blocks(const Layout &L);
cudaError_t configure_kernels();
// device address (on the current device) and capacity, in reduction CTAs, of the static scratch of clt_diagnostics_static
cudaError_t diag_static_scratch(double **ptr, int *max_blocks);

}  // namespace clt
