// clt_kernels.cu -- sm_100a CUDA kernels of libclt (product code; shares nothing with oracle/).
//
// Hot path ("DERIVATIVES", "J, E", "RIGHT HANDS OF EQUATIONS", "STEP ON"):
//   curl_kernel : J1 = curl_c(B - B0)                                   (eq 6)
//   rhs_kernel  : E1, all derivatives, K of eqs (11)-(14) (L105-115) and the RK4 stage combine in
//                 the epilogue, one read and one write of HBM per stage.
// Both are 2.5-D sweeps: a CTA owns a TR x TZ tile of the (R, Z) plane and marches along phi;
// in-plane neighbours come from a shared-memory tile with a radius-2 halo, phi neighbours from a
// 5-deep register pipeline (rho1, p1, v1) and from shared-memory rings (E1, J x B force).
// Everything differenced is a perturbation (U - U0): DESIGN.md section 3, hazard H2.
#include "clt_internal.h"
#include <cuda.h>

namespace clt {

// launch shape of curl_tma_kernel: tile height, ring depth (planes), CTAs per SM
#ifndef CLT_CURL_TZ
#define CLT_CURL_TZ 10
#define CLT_CURL_NS 6
#define CLT_CURL_MINB 2
#endif
// outputs per thread (= width of the sliding register windows) of the pseudo-spectral pre-pass
#ifndef CLT_SPEC_NQ
#define CLT_SPEC_NQ 8
#endif

constexpr int TR = 32;        // tile width in R = one warp per tile row
constexpr int SW = TR + 4;    // shared row width with the radius-2 halo

__device__ __forceinline__ void prefetch_l2(const void *p)
{
    asm volatile("prefetch.global.L2 [%0];" ::"l"(p));
}

// unscaled 4th-order central differences from five equally spaced samples:
//   d1 * 1/(12h)   = first derivative,  d2 * 1/(12h^2) = second derivative
__device__ __forceinline__ double fd1(double m2, double m1, double p1, double p2)
{
    return 8.0 * (p1 - m1) - (p2 - m2);
}
__device__ __forceinline__ double fd2(double m2, double m1, double c0, double p1, double p2)
{
    return (16.0 * (p1 + m1) - (p2 + m2)) - 30.0 * c0;
}

__device__ __forceinline__ int wrap_phi(int j, int n)
{
    return j < 0 ? j + n : (j >= n ? j - n : j);
}

// ---------------------------------------------------------------------------------------------
// a3-a5 at one node: K of eqs (11)-(14) from
//   stg  [2][HT]    centre-plane tile (with halo) of rho1, p1; field f at stg + f*HT
//   stgV [3][HT]    centre-plane tile (with halo) of v1_R, v1_phi, v1_Z (the TMA-fed kernel with a static reference state
//                   reads the velocity tiles as they arrived: v1 = v)
//   eRc, ePc, eZc   E1_R / E1_phi / E1_Z tiles (with halo) of the centre plane
//   dP_EZ, dP_ER    unscaled phi differences (fd1) of E1_Z, E1_R at the own node
//   F    [3]        J1 x B + J0 x B1 at the own node of the centre plane
//   rr   [4]        R_{i-2}, R_{i-1}, R_{i+1}, R_{i+2}
//   q    [5][5]     phi pipeline of the five fluid perturbations at this node, planes j-2..j+2
// ---------------------------------------------------------------------------------------------
// axisymmetric table values of one node that the centre-plane arithmetic needs (phi-invariant, so a
// thread can keep them in registers for the whole sweep)
struct CentreTab {
    double rho0, p0, gRrho0, gZrho0, gRp0, gZp0;
};
__device__ __forceinline__ CentreTab load_centre_tab(const double *tab, long long plane, long long off2)
{
    CentreTab t;
    t.rho0 = __ldg(tab + T_RHO0 * plane + off2);
    t.p0 = __ldg(tab + T_P0 * plane + off2);
    t.gRrho0 = __ldg(tab + T_GR_RHO0 * plane + off2);
    t.gZrho0 = __ldg(tab + T_GZ_RHO0 * plane + off2);
    t.gRp0 = __ldg(tab + T_GR_P0 * plane + off2);
    t.gZp0 = __ldg(tab + T_GZ_P0 * plane + off2);
    return t;
}

// `sync` is called once, after everything that needs no other thread's shared-memory data (centre values, the
// phi direction from the register pipeline, the phi differences of E1 at the own node) and before the first read
// of a neighbour's staged value: the caller puts the wait half of its split barrier there.
// SPEC = true: the phi derivatives come from the pseudo-spectral pre-pass: pd1[f], pd2[f] are d/dphi and d2/dphi2 of
// the five fluid perturbations, dP_EZ / dP_ER the true d/dphi of E1_Z / E1_R (not the unscaled stencil sums).
template <bool V0, bool SPEC, class Sync>
__device__ __forceinline__ void rhs_point(const double *stg, const double *stgV, int HT, const double *eRc, const double *ePc, const double *eZc,
                                          double dP_EZ, double dP_ER, const double (&F)[3], const double (&rr)[4], int cs,
                                          const double (&q)[5][5], const CentreTab &ct, const double *tab, long long off2,
                                          long long plane, const Phys &ph, double iR, double iR2, double (&K)[8], Sync &&sync,
                                          const double *pd1 = nullptr, const double *pd2 = nullptr)
{
    const double rho1 = q[2][0], p1 = q[2][1], v1R = q[2][2], v1P = q[2][3], v1Z = q[2][4];
    const double rho = rho1 + ct.rho0;
    const double p = p1 + ct.p0;
    double vR = v1R, vP = v1P, vZ = v1Z;
    if (V0) {
        vR += __ldg(tab + T_V0R * plane + off2);
        vP += __ldg(tab + T_V0P * plane + off2);
        vZ += __ldg(tab + T_V0Z * plane + off2);
    }
    const double rinv = 1.0 / rho;

    double A[5], lap[5];     // (v.grad) f and Laplacian f of the five staged fields
    double divv1, gRp1, gPp1, gZp1, gPvR, gPvP;
    // phi direction (register pipeline)
    {
        const double g1 = SPEC ? iR : ph.cP1 * iR, vc = vP * g1, lc = SPEC ? iR2 : ph.cP2 * iR2;
#pragma unroll
        for (int f = 0; f < 5; ++f) {
            const double d1 = SPEC ? pd1[f] : fd1(q[0][f], q[1][f], q[3][f], q[4][f]);
            const double d2 = SPEC ? pd2[f] : fd2(q[0][f], q[1][f], q[2][f], q[3][f], q[4][f]);
            A[f] = vc * d1;
            lap[f] = lc * d2;
            if (f == 1) gPp1 = d1 * g1;
            if (f == 2) gPvR = d1 * g1;
            if (f == 3) { gPvP = d1 * g1; divv1 = gPvP + v1R * iR; }
        }
    }
    const double fR = F[0], fP = F[1], fZ = F[2];

    sync();

    // R direction (shared memory, stride 1)
    {
        const double vc = vR * ph.cR1, lc = iR * ph.cR1;
#pragma unroll
        for (int f = 0; f < 5; ++f) {
            const double *s = (f < 2 ? stg + f * HT : stgV + (f - 2) * HT) + cs;
            const double m2 = s[-2], m1 = s[-1], p1_ = s[1], p2 = s[2];
            const double d1 = fd1(m2, m1, p1_, p2), d2 = fd2(m2, m1, q[2][f], p1_, p2);
            A[f] += vc * d1;
            lap[f] += d2 * ph.cR2 + lc * d1;
            if (f == 1) gRp1 = d1 * ph.cR1;
            if (f == 2) divv1 += d1 * ph.cR1;
        }
    }
    // Z direction (shared memory, stride SW)
    {
        const double vc = vZ * ph.cZ1;
#pragma unroll
        for (int f = 0; f < 5; ++f) {
            const double *s = (f < 2 ? stg + f * HT : stgV + (f - 2) * HT) + cs;
            const double m2 = s[-2 * SW], m1 = s[-SW], p1_ = s[SW], p2 = s[2 * SW];
            const double d1 = fd1(m2, m1, p1_, p2), d2 = fd2(m2, m1, q[2][f], p1_, p2);
            A[f] += vc * d1;
            lap[f] += d2 * ph.cZ2;
            if (f == 1) gZp1 = d1 * ph.cZ1;
            if (f == 4) divv1 += d1 * ph.cZ1;
        }
    }

    // eq (11), L105 and eq (12), with grad rho = grad rho1 + grad rho0 (tables)
    double cr = A[0] + v1R * ct.gRrho0 + v1Z * ct.gZrho0 + rho * divv1;
    double cp = A[1] + v1R * ct.gRp0 + v1Z * ct.gZp0;
    double pd = p * divv1;
    if (V0) {
        const double dv0 = __ldg(tab + T_DIVV0 * plane + off2);
        cr += rho1 * dv0;
        pd += p1 * dv0;
    }
    K[0] = ph.D * lap[0] - cr;
    K[1] = ph.kappa * lap[1] - cp - ph.gamma * pd;
    // eq (13)
    double aR = A[2] - vP * v1P * iR;
    double aP = A[3] + vP * v1R * iR;
    double aZ = A[4];
    if (V0) {
        const double v0R = vR - v1R, v0P = vP - v1P;
        const double r1 = rho1 * rinv;
        aR += v1R * __ldg(tab + T_GR_V0R * plane + off2) + v1Z * __ldg(tab + T_GZ_V0R * plane + off2)
              - v1P * v0P * iR + r1 * __ldg(tab + T_A0R * plane + off2);
        aP += v1R * __ldg(tab + T_GR_V0P * plane + off2) + v1Z * __ldg(tab + T_GZ_V0P * plane + off2)
              + v1P * v0R * iR + r1 * __ldg(tab + T_A0P * plane + off2);
        aZ += v1R * __ldg(tab + T_GR_V0Z * plane + off2) + v1Z * __ldg(tab + T_GZ_V0Z * plane + off2)
              + r1 * __ldg(tab + T_A0Z * plane + off2);
    }
    const double two_iR = 2.0 * iR;
    K[2] = (fR - gRp1) * rinv - aR + ph.nu * (lap[2] - v1R * iR2 - two_iR * gPvP);
    K[3] = (fP - gPp1) * rinv - aP + ph.nu * (lap[3] - v1P * iR2 + two_iR * gPvR);
    K[4] = (fZ - gZp1) * rinv - aZ + ph.nu * lap[4];
    // eq (14): -curl_c(E1); the radial derivative differences R * E_phi
    const double *eR = eRc + cs, *eP = ePc + cs, *eZ = eZc + cs;
    const double dZ_EP = fd1(eP[-2 * SW], eP[-SW], eP[SW], eP[2 * SW]);
    const double dZ_ER = fd1(eR[-2 * SW], eR[-SW], eR[SW], eR[2 * SW]);
    const double dR_EZ = fd1(eZ[-2], eZ[-1], eZ[1], eZ[2]);
    const double dR_REP = fd1(rr[0] * eP[-2], rr[1] * eP[-1], rr[2] * eP[1], rr[3] * eP[2]);
    const double cPi = SPEC ? iR : ph.cP1 * iR;
    K[5] = dZ_EP * ph.cZ1 - dP_EZ * cPi;
    K[6] = dR_EZ * ph.cR1 - dZ_ER * ph.cZ1;
    K[7] = dP_ER * cPi - dR_REP * (ph.cR1 * iR);
}

// ---------------------------------------------------------------------------------------------
// a6: RK4 stage combine (L125, L139) in a reduced-traffic accumulator form.
// Classical RK4, U^{n+1} = U^n + dt/6 (K1 + 2 K2 + 2 K3 + K4).  The accumulator holds the INCREMENT
// dt/6 K1 + dt/3 K2 (+ ...), never the state: U^n is added once, in stage 4, so a step rounds the state once at the
// size of U -- like the literal formula above -- instead of once per stage (for B_phi ~ 1 next to v_phi ~ 1e-7 every
// extra rounding of the state is visible in v_phi after 100 steps: DESIGN.md reading R10).  The partial sums are
// rebuilt from stage states that are read anyway instead of being written and re-read through a separate array:
//   S1: U_a = U^n + dt/2 K1                                        (no accumulator write)
//   S2: U_b = U^n + dt/2 K2,  acc = (U_a - U^n)/3 + dt/3 K2         ((U_a - U^n)/3 = dt/6 K1)
//   S3: U_a = U^n + dt K3                                          (no accumulator traffic)
//   S4: U^{n+1} = U^n + [acc + (U_a - U^n)/3 + dt/6 K4]             ((U_a - U^n)/3 = dt/3 K3)
// Identical to the textbook scheme up to rounding order.  Per node and step this moves 19 + 35 + 27 + 35
// doubles through the fused kernel instead of 27 + 43 + 43 + 27.
// -DCLT_TEXTBOOK_RK4 builds the textbook accumulator schedule instead (libclt_textbook.so; the A/B that shows what
// the reduced schedule costs in round-off -- BASELINE.md section 4 -- never the product's default):
//   S1: U_a = U^n + dt/2 K1, acc = dt/6 K1            S2: U_b = U^n + dt/2 K2, acc += dt/3 K2
//   S3: U_a = U^n + dt K3,   acc += dt/3 K3           S4: U^{n+1} = U^n + (acc + dt/6 K4)
// ---------------------------------------------------------------------------------------------
#ifdef CLT_TEXTBOOK_RK4
constexpr bool TEXTBOOK_RK4 = true;
#else
constexpr bool TEXTBOOK_RK4 = false;
#endif
__device__ __forceinline__ void st_out(double *p, double v) { *p = v; }

struct EpiOperands {
    double un[8];   // U^n at the node
    double us[8];   // stage state at the node (S2: U_a of stage 1, S4: U_a of stage 3)
    double ac[8];   // accumulator (S4)
};
// NOWN > 0: the caller still holds the first NOWN fields of the stage state at this node (own[m]; rho, p[, v]
// rebuilt as perturbation + reference value, exact whenever the perturbation was formed exactly) and they are
// taken from there instead of being read again.
template <int MODE, int NOWN, class Load>
__device__ __forceinline__ void epilogue_load(const RhsArgs &a, long long g, long long field, EpiOperands &e, Load &&ld,
                                              const double *own = nullptr)
{
#pragma unroll
    for (int m = 0; m < 8; ++m) {
        const long long gm = m * field + g;
        if (MODE == RHS_MODE_S1) e.un[m] = (m < NOWN) ? own[m] : ld(a.in + gm);
        if (TEXTBOOK_RK4) {
            if (MODE == RHS_MODE_S2 || MODE == RHS_MODE_S3 || MODE == RHS_MODE_S4) {
                e.un[m] = ld(a.Un + gm);
                e.ac[m] = ld(a.acc + gm);
            }
            continue;
        }
        if (MODE == RHS_MODE_S2 || MODE == RHS_MODE_S3 || MODE == RHS_MODE_S4) e.un[m] = ld(a.Un + gm);
        if (MODE == RHS_MODE_S2 || MODE == RHS_MODE_S4) e.us[m] = (m < NOWN) ? own[m] : ld(a.in + gm);
        if (MODE == RHS_MODE_S4) e.ac[m] = ld(a.acc + gm);
    }
}
// The stage coefficients come from device memory (a.coef = { dt, dt/2, dt/3, dt/6 }: the fixed-dt table, or the clock
// that dt_commit_kernel advances).  Adaptive stepping (clt_step_cfl, NEXT-1): stage 4 folds the SETDT minimum of the
// new state into `rate` (Fig. 3: STEPON then SETDT, without a separate pass over the state).
// out = U^n + an K (stages 1-3: dt/2, dt/2, dt); bn = weight of K in the accumulator (stage 2: dt/3) / in U^{n+1}
// (stage 4: dt/6).  Read once per thread, before the sweep.
struct StageCoef {
    double an, bn;
};
template <int MODE>
__device__ __forceinline__ StageCoef load_stage_coef(const RhsArgs &a)
{
    StageCoef c = { 0.0, 0.0 };
    if (MODE != RHS_MODE_K) {
        c.an = __ldg(a.coef + (MODE == RHS_MODE_S3 ? 0 : 1));
        c.bn = __ldg(a.coef + ((MODE == RHS_MODE_S2 || (TEXTBOOK_RK4 && MODE == RHS_MODE_S3)) ? 2 : 3));
    }
    return c;
}
template <int MODE>
__device__ __forceinline__ void epilogue_store(const RhsArgs &a, long long g, long long field, const EpiOperands &e,
                                               const double (&K)[8], double iR, double &rate, const StageCoef &sc, bool collect,
                                               double *peer0 = nullptr, double *peer1 = nullptr)
{
    constexpr double third = 1.0 / 3.0;
    const double an = sc.an, bn = sc.bn;
    double out[8];
    // the stage's output at this node; peer0 / peer1: the same node in a neighbouring slab's buffer (its ghost row), or null
    auto put = [&](int m, double v) {
        st_out(a.out + m * field + g, v);
        if (MODE != RHS_MODE_K) {
            if (peer0) st_out(peer0 + m * a.peer[0].field, v);
            if (peer1) st_out(peer1 + m * a.peer[1].field, v);
        }
    };
#pragma unroll
    for (int m = 0; m < 8; ++m) {
        const long long gm = m * field + g;
        if (MODE == RHS_MODE_K) {
            put(m, K[m]);
        } else if (TEXTBOOK_RK4) {
            if (MODE == RHS_MODE_S1) {
                put(m, fma(an, K[m], e.un[m]));
                st_out(a.acc + gm, bn * K[m]);
            } else if (MODE == RHS_MODE_S2 || MODE == RHS_MODE_S3) {
                put(m, fma(an, K[m], e.un[m]));
                st_out(a.acc + gm, fma(bn, K[m], e.ac[m]));
            } else {
                out[m] = e.un[m] + fma(bn, K[m], e.ac[m]);
                put(m, out[m]);
            }
        } else if (MODE == RHS_MODE_S1 || MODE == RHS_MODE_S3) {
            put(m, fma(an, K[m], e.un[m]));
        } else if (MODE == RHS_MODE_S2) {
            put(m, fma(an, K[m], e.un[m]));
            st_out(a.acc + gm, fma(bn, K[m], (e.us[m] - e.un[m]) * third));
        } else {
            out[m] = e.un[m] + fma(bn, K[m], fma(e.us[m] - e.un[m], third, e.ac[m]));
            put(m, out[m]);
        }
    }
    if (MODE == RHS_MODE_S4 && a.dtmin_bits && collect) {
        // SETDT of Fig. 4 regrouped (rounding order only): dt = cfl / max_d (|v_d| + c) / h_d with the uniform spacings
        // 1/dR = 12 cR1, 1/dZ = 12 cZ1, 1/(R dphi) = 12 cP1 / R; one division and one square root per node here, the
        // division by the largest rate once per thread in dtmin_commit
        const double b2 = out[5] * out[5] + out[6] * out[6] + out[7] * out[7];
        const double cf = sqrt(fabs((a.ph.gamma * out[1] + b2) / out[0]));
        const double rR = (fabs(out[2]) + cf) * a.ph.cR1, rP = (fabs(out[3]) + cf) * (a.ph.cP1 * iR),
                     rZ = (fabs(out[4]) + cf) * a.ph.cZ1;
        rate = fmax(rate, fmax(rP, fmax(rR, rZ)));
        // fmax drops NaN: a non-finite new state must not pass for "no signal" (dt = 100).  An infinite rate gives
        // dt = 0, which dt_commit_kernel turns into the clock's non-finite mark and clt_step_cfl into CLT_ENONFINITE.
        if (!(rR + rP + rZ <= 1.79769313486231570815e308)) rate = __longlong_as_double(0x7ff0000000000000LL);
    }
}

// the node (i, k, plane j) in the buffer of neighbouring slab `side`, if row k is one of the rows it takes from us
__device__ __forceinline__ double *peer_node(const RhsArgs &a, int side, int i, int k, int j, int pR)
{
    const RhsArgs::Peer &p = a.peer[side];
    if (!p.out || k < p.k0 || k > p.k1) return nullptr;
    return p.out + (long long)j * p.plane + (long long)(k + p.dk) * pR + (LP + i);
}

// end of a stage-4 kernel: this thread's largest signal rate -> its SETDT value -> device-wide minimum (positive doubles
// order like their bit patterns)
__device__ __forceinline__ void dtmin_commit(const RhsArgs &a, double rate)
{
    if (!a.dtmin_bits) return;
    double dtmin = rate > 0.0 ? a.cfl / (12.0 * rate) : 100.0;
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) dtmin = fmin(dtmin, __shfl_xor_sync(0xffffffffu, dtmin, o));
    if ((threadIdx.x & 31) == 0) atomicMin(a.dtmin_bits, (unsigned long long)__double_as_longlong(dtmin));
}

// one thread: opens (init = 1: dt from the SETDT reduction `diag6[5]`, time = 0) or advances (time += dt just used,
// dt = the minimum stage 4 collected) the device-side clock of clt_step_cfl.
// clock = { dt, dt/2, dt/3, dt/6, time, non-finite mark }.  A state with a non-finite signal speed yields dt = 0 (stage 4) or
// a NaN / non-positive SETDT value (init): the mark is raised, dt stays 0 (the remaining steps of the call change
// nothing) and clt_step_cfl returns CLT_ENONFINITE.
__global__ void dt_commit_kernel(double *clock, unsigned long long *dtmin_bits, const double *diag6, int init)
{
    double dt;
    if (init) {
        dt = diag6[5];
        clock[4] = 0.0;
        clock[5] = 0.0;
    } else {
        clock[4] += clock[0];
        dt = fmin(100.0, __longlong_as_double((long long)*dtmin_bits));
    }
    if (!(dt > 0.0) || clock[5] != 0.0) {
        clock[5] = 1.0;
        dt = 0.0;
    }
    clock[0] = dt; clock[1] = 0.5 * dt; clock[2] = dt / 3.0; clock[3] = dt / 6.0;
    *dtmin_bits = (unsigned long long)__double_as_longlong(100.0);      // Fig. 4: DT1 starts at 100
}

// The same for a group of contexts that share one time step (slabs of one grid): the minimum over all of them goes to
// every clock.
__global__ void dt_commit_group_kernel(DtGroup g, int init)
{
    double dt = 100.0;
    bool marked = false;
    for (int c = 0; c < g.n; ++c) {
        const double mine = init ? g.diag6[c][5] : __longlong_as_double((long long)*g.dtmin_bits[c]);
        if (!(mine > 0.0)) marked = true;
        dt = fmin(dt, mine);
        if (!init && g.clock[c][5] != 0.0) marked = true;
    }
    if (marked) dt = 0.0;
    for (int c = 0; c < g.n; ++c) {
        double *clock = g.clock[c];
        if (init) clock[4] = 0.0; else clock[4] += clock[0];
        clock[5] = marked ? 1.0 : 0.0;
        clock[0] = dt; clock[1] = 0.5 * dt; clock[2] = dt / 3.0; clock[3] = dt / 6.0;
        *g.dtmin_bits[c] = (unsigned long long)__double_as_longlong(100.0);
    }
}

cudaError_t launch_dt_commit_group(const DtGroup &g, int init, cudaStream_t s)
{
    dt_commit_group_kernel<<<1, 1, 0, s>>>(g, init);
    return cudaGetLastError();
}

cudaError_t launch_dt_commit(double *clock, unsigned long long *dtmin_bits, const double *diag6, int init, cudaStream_t s)
{
    dt_commit_kernel<<<1, 1, 0, s>>>(clock, dtmin_bits, diag6, init);
    return cudaGetLastError();
}

// ---------------------------------------------------------------------------------------------
// Fused RHS + RK4 stage combine
// ---------------------------------------------------------------------------------------------
template <int TZ>
struct RhsSmem {
    static constexpr int HT = (TZ + 4) * SW;   // tile with halo
    static constexpr int IT = TZ * TR;         // tile interior
    double stage[2][5][HT];    // rho1, p1, v1_R, v1_phi, v1_Z of the centre plane (double-buffered)
    double ering[5][3][HT];    // E1 of planes j-2 .. j+2 (halo part valid for the centre plane only)
    double fring[3][3][IT];    // F = J1 x B + J0 x B1 of planes j .. j+2
    double sR[SW];             // R_i of the tile columns i0-2 .. i0+33
};

template <int TZ, int MODE, bool V0>
__global__ void __launch_bounds__(TR *TZ, 1) rhs_kernel(const __grid_constant__ RhsArgs a)
{
    extern __shared__ __align__(128) unsigned char smem_raw[];
    RhsSmem<TZ> &S = *reinterpret_cast<RhsSmem<TZ> *>(smem_raw);
    const Layout &L = a.L;
    const Phys &ph = a.ph;

    const int tx = threadIdx.x, ty = threadIdx.y, tid = ty * TR + tx;
    const int i0 = 2 + TR * blockIdx.x, k0 = 2 + TZ * blockIdx.y;
    const int i = i0 + tx, k = k0 + ty;
    // a stage writes the context's owned rows only (clt_rhs: every interior row)
    const bool valid = (i <= L.nR - 3) && (k <= L.nZ - 3) && (MODE == RHS_MODE_K || (k >= a.own_k0 && k <= a.own_k1));
    const int ic = min(i, L.nR - 1), kc = min(k, L.nZ - 1);
    const int ja = (int)(((long long)L.nphi * blockIdx.z) / a.phi_chunks);
    const int jb = (int)(((long long)L.nphi * (blockIdx.z + 1)) / a.phi_chunks);

    const long long off2 = (long long)kc * L.pR + (LP + ic);     // offset inside a plane / a table
    const int cs = (ty + 2) * SW + (tx + 2);                     // own slot in a halo tile
    const int ci = ty * TR + tx;                                 // own slot in an interior tile

    // halo nodes: 4 full rows (Z halo) then 4 columns (R halo); one node per thread, tid < NH
    constexpr int NH = 4 * TR + 4 * TZ;
    static_assert(NH <= TR * TZ, "tile too small for one halo node per thread");
    int hx, hy;
    if (tid < 4 * TR) {
        const int r = tid / TR;
        hx = tid % TR;
        hy = (r < 2) ? r - 2 : TZ + (r - 2);
    } else {
        const int t = tid - 4 * TR, c = t & 3;
        hy = t >> 2;
        hx = (c < 2) ? c - 2 : TR + (c - 2);
    }
    const bool is_halo = tid < NH;
    const int hi = min(i0 + hx, L.nR - 1), hk = min(k0 + hy, L.nZ - 1);
    const long long hoff2 = (long long)hk * L.pR + (LP + hi);
    const int hs = (hy + 2) * SW + (hx + 2);

    if (tid < SW) S.sR[tid] = a.R[min(i0 - 2 + tid, L.nR - 1)];

    const double *tab = a.tab;
    const double eta = ph.eta;

    // loads the 11 stage fields at one node of one plane, forms perturbations, E1 and (optionally) F
    auto load_node = [&](long long o2, int jw, double q[5], double E[3], double F[3], bool wantF) {
        const long long g = (long long)jw * L.plane + o2;
        const double rho = __ldg(a.in + 0 * L.field + g), p = __ldg(a.in + 1 * L.field + g);
        const double vR = __ldg(a.in + 2 * L.field + g), vP = __ldg(a.in + 3 * L.field + g),
                     vZ = __ldg(a.in + 4 * L.field + g);
        const double BR = __ldg(a.in + 5 * L.field + g), BP = __ldg(a.in + 6 * L.field + g),
                     BZ = __ldg(a.in + 7 * L.field + g);
        const double JR = __ldg(a.J1 + 0 * L.field + g), JP = __ldg(a.J1 + 1 * L.field + g),
                     JZ = __ldg(a.J1 + 2 * L.field + g);
        q[0] = rho - __ldg(tab + T_RHO0 * L.plane + o2);
        q[1] = p - __ldg(tab + T_P0 * L.plane + o2);
        if (V0) {
            q[2] = vR - __ldg(tab + T_V0R * L.plane + o2);
            q[3] = vP - __ldg(tab + T_V0P * L.plane + o2);
            q[4] = vZ - __ldg(tab + T_V0Z * L.plane + o2);
        } else {
            q[2] = vR; q[3] = vP; q[4] = vZ;
        }
        // a4: E1 = -v x B + v0 x B0 + eta J1   (eq 5 with d_i = 0 minus E0, L77, L101)
        E[0] = eta * JR - (vP * BZ - vZ * BP);
        E[1] = eta * JP - (vZ * BR - vR * BZ);
        E[2] = eta * JZ - (vR * BP - vP * BR);
        if (V0) {
            E[0] += __ldg(tab + T_E0R * L.plane + o2);
            E[1] += __ldg(tab + T_E0P * L.plane + o2);
            E[2] += __ldg(tab + T_E0Z * L.plane + o2);
        }
        if (wantF) {
            const double B1R = BR - __ldg(tab + T_B0R * L.plane + o2), B1P = BP - __ldg(tab + T_B0P * L.plane + o2),
                         B1Z = BZ - __ldg(tab + T_B0Z * L.plane + o2);
            const double J0R = __ldg(tab + T_J0R * L.plane + o2), J0P = __ldg(tab + T_J0P * L.plane + o2),
                         J0Z = __ldg(tab + T_J0Z * L.plane + o2);
            // Lorentz force terms of eq (13): J1 x B + J0 x B1
            F[0] = (JP * BZ - JZ * BP) + (J0P * B1Z - J0Z * B1P);
            F[1] = (JZ * BR - JR * BZ) + (J0Z * B1R - J0R * B1Z);
            F[2] = (JR * BP - JP * BR) + (J0R * B1P - J0P * B1R);
        }
    };

    double q[5][5];      // phi pipeline: q[d][f], plane j-2+d, f = rho1, p1, v1R, v1P, v1Z
    int se = 0, sf = 0;  // ring slots that receive plane j+2

    auto lead = [&](int jl) {
        double E[3], F[3];
        load_node(off2, wrap_phi(jl, L.nphi), q[4], E, F, true);
#pragma unroll
        for (int c = 0; c < 3; ++c) {
            S.ering[se][c][cs] = E[c];
            S.fring[sf][c][ci] = F[c];
        }
    };
    auto advance = [&]() {
#pragma unroll
        for (int d = 0; d < 4; ++d)
#pragma unroll
            for (int f = 0; f < 5; ++f) q[d][f] = q[d + 1][f];
        se = (se == 4) ? 0 : se + 1;
        sf = (sf == 2) ? 0 : sf + 1;
    };

    // prologue: planes ja-2 .. ja+1
#pragma unroll 1
    for (int jl = ja - 2; jl <= ja + 1; ++jl) {
        lead(jl);
        advance();
    }

    const double iR = __ldg(a.invR + ic);
    const double iR2 = iR * iR;
    double rate = 0.0;           // largest signal rate (|v_d| + c)/(12 h_d) at this thread's nodes (stage 4 of clt_step_cfl)
    const StageCoef coef = load_stage_coef<MODE>(a);

#pragma unroll 1
    for (int j = ja; j < jb; ++j) {
        const int buf = j & 1;
        const int jw = j;   // ja <= j < jb <= nphi: no wrap needed for the centre plane
        // ---- phase A: stage plane j, bring in plane j+2 --------------------------------------
        if (a.prefetch && (tx & 15) == 0) {
            const long long g3 = (long long)wrap_phi(j + 3, L.nphi) * L.plane + off2;
#pragma unroll
            for (int m = 0; m < 8; ++m) prefetch_l2(a.in + m * L.field + g3);
#pragma unroll
            for (int m = 0; m < 3; ++m) prefetch_l2(a.J1 + m * L.field + g3);
            if (MODE != RHS_MODE_K && j + 1 < jb) {
                const long long g1 = (long long)(j + 1) * L.plane + off2;
#pragma unroll
                for (int m = 0; m < 8; ++m) {
                    if (MODE != RHS_MODE_S1) prefetch_l2(a.Un + m * L.field + g1);
                    if (MODE == RHS_MODE_S4) prefetch_l2(a.acc + m * L.field + g1);
                }
            }
        }
        lead(j + 2);
#pragma unroll
        for (int f = 0; f < 5; ++f) S.stage[buf][f][cs] = q[2][f];
        const int sec = (se + 3 >= 5) ? se + 3 - 5 : se + 3;      // ring slot of the centre plane
        if (is_halo) {
            double hq[5], hE[3], hF[3];
            load_node(hoff2, jw, hq, hE, hF, false);
#pragma unroll
            for (int f = 0; f < 5; ++f) S.stage[buf][f][hs] = hq[f];
#pragma unroll
            for (int c = 0; c < 3; ++c) S.ering[sec][c][hs] = hE[c];
        }
        __syncthreads();

        // ---- phase B: K at (i, k, j) -----------------------------------------------------------
        double K[8];
        {
            const int sfc = (sf + 1 >= 3) ? sf + 1 - 3 : sf + 1;  // ring slot of F at the centre plane
            const CentreTab ct = load_centre_tab(tab, L.plane, off2);
            // phi differences of E1_Z, E1_R at the own node (ring slots written by this very thread):
            // slot se = plane j+2, so j-2 -> se+1, j-1 -> se+2, j+1 -> se+4 (mod 5)
            const int s0 = (se + 1 >= 5) ? se + 1 - 5 : se + 1, s1 = (se + 2 >= 5) ? se + 2 - 5 : se + 2;
            const int s3 = (se + 4 >= 5) ? se + 4 - 5 : se + 4;
            const double dP_EZ = fd1(S.ering[s0][2][cs], S.ering[s1][2][cs], S.ering[s3][2][cs], S.ering[se][2][cs]);
            const double dP_ER = fd1(S.ering[s0][0][cs], S.ering[s1][0][cs], S.ering[s3][0][cs], S.ering[se][0][cs]);
            const double F[3] = { S.fring[sfc][0][ci], S.fring[sfc][1][ci], S.fring[sfc][2][ci] };
            const double rr[4] = { S.sR[tx], S.sR[tx + 1], S.sR[tx + 3], S.sR[tx + 4] };
            rhs_point<V0, false>(&S.stage[buf][0][0], &S.stage[buf][2][0], RhsSmem<TZ>::HT, &S.ering[sec][0][0], &S.ering[sec][1][0], &S.ering[sec][2][0],
                          dP_EZ, dP_ER, F, rr, cs, q, ct, tab, off2, L.plane, ph, iR, iR2, K, [] {});
        }

        // ---- a6: RK4 stage combine in the epilogue (L125, L139) --------------------------------
        if (valid) {
            const long long g = (long long)jw * L.plane + off2;
            EpiOperands eo;
            // plain coherent loads: stage 4 updates U^n in place through a.out, so the non-coherent path is not allowed here
            epilogue_load<MODE, 0>(a, g, L.field, eo, [](const double *p) { return *p; });
            epilogue_store<MODE>(a, g, L.field, eo, K, iR, rate, coef, true);
        }
        advance();
    }
    if (MODE == RHS_MODE_S4) dtmin_commit(a, rate);
}

// configure = true: only opt the kernel in to its dynamic shared-memory size on the current device (clt_create)
template <int TZ, int MODE, bool V0>
static cudaError_t launch_rhs_t(const RhsArgs &a, cudaStream_t s, bool configure)
{
    auto kern = rhs_kernel<TZ, MODE, V0>;
    const int smem = (int)sizeof(RhsSmem<TZ>);
    if (configure) return cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, smem);
    dim3 block(TR, TZ, 1);
    dim3 grid((a.L.nR - 4 + TR - 1) / TR, (a.L.nZ - 4 + TZ - 1) / TZ, a.phi_chunks);
    kern<<<grid, block, smem, s>>>(a);
    return cudaGetLastError();
}

constexpr int RHS_TZ = 8;     // tile height of both fused-kernel variants (32 x 8 nodes, one node per thread)
int rhs_tile_z() { return RHS_TZ; }

// plain-load variant (variant 1): the A/B and parity cross-check of the TMA-fed default
cudaError_t launch_rhs(const RhsArgs &a, int mode, bool has_v0, cudaStream_t s, bool configure)
{
#define CLT_CASE(M)                                                      \
    case M:                                                              \
        return has_v0 ? launch_rhs_t<RHS_TZ, M, true>(a, s, configure) : launch_rhs_t<RHS_TZ, M, false>(a, s, configure);
    switch (mode) {
        CLT_CASE(RHS_MODE_K)
        CLT_CASE(RHS_MODE_S1)
        CLT_CASE(RHS_MODE_S2)
        CLT_CASE(RHS_MODE_S3)
        CLT_CASE(RHS_MODE_S4)
    default:
        return cudaErrorInvalidValue;
    }
#undef CLT_CASE
}

// ---------------------------------------------------------------------------------------------
// TMA variant of the fused RHS kernel (the default).  Same arithmetic (rhs_point), but the 11 stage
// fields of plane j+3 arrive as halo'd (TR+4) x (TZ+4) boxes through cp.async.bulk.tensor into one
// shared "raw" buffer while plane j is being computed, completing on an mbarrier: the long-latency
// HBM/L2 reads never sit in front of the FP64 work and cost no registers.  Every plane is read from
// L2 exactly once per CTA (interior + halo in one box) and converted once, on arrival, into the
// perturbations and E1 that the stencils need (4-slot shared rings, tile with halo); everything that only
// the own node needs along phi (fluid pipeline, E1_R/E1_Z pipeline, the Lorentz term F, R neighbours)
// lives in registers: shared-memory bandwidth is the second roof of this kernel.
// ---------------------------------------------------------------------------------------------
// streaming 8-byte load that does not allocate in L1 (the epilogue operands are touched exactly once);
// volatile so that it is issued where it is written: ahead of the FP64 work that hides its latency
__device__ __forceinline__ double ld_stream(const double *p)
{
    double v;
    asm volatile("ld.global.L1::no_allocate.f64 %0, [%1];" : "=d"(v) : "l"(p) : "memory");
    return v;
}

__device__ __forceinline__ unsigned smem_u32(const void *p) { return (unsigned)__cvta_generic_to_shared(p); }

__device__ __forceinline__ void mbar_init(unsigned long long *bar, unsigned count)
{
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(bar)), "r"(count));
}
__device__ __forceinline__ void mbar_expect_tx(unsigned long long *bar, unsigned bytes)
{
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(bar)), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_arrive(unsigned long long *bar)
{
    asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(smem_u32(bar)) : "memory");
}
__device__ __forceinline__ void mbar_wait(unsigned long long *bar, unsigned parity)
{
    asm volatile(
        "{\n"
        ".reg .pred p;\n"
        "WAIT_LOOP:\n"
        "mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n"
        "@p bra.uni WAIT_DONE;\n"
        "bra.uni WAIT_LOOP;\n"
        "WAIT_DONE:\n"
        "}\n" ::"r"(smem_u32(bar)), "r"(parity) : "memory");
}
__device__ __forceinline__ void tma_load_4d(void *dst, const CUtensorMap *map, int c0, int c1, int c2, int c3,
                                            unsigned long long *bar)
{
    // L2 evict_last on the tiles: every halo row / column is read again by the neighbouring tile's CTA a little later,
    // the epilogue operands and outputs that stream through L2 next to them are not (measured: -2 % on the HBM-bound
    // stage 2 and on the curl kernel; evict_first hints on the epilogue loads / stores change nothing)
    unsigned long long pol;
    asm volatile("createpolicy.fractional.L2::evict_last.b64 %0, 1.0;" : "=l"(pol));
    asm volatile(
        "cp.async.bulk.tensor.4d.shared::cluster.global.mbarrier::complete_tx::bytes.L2::cache_hint [%0], [%1, {%2, %3, %4, %5}], [%6], %7;" ::"r"(
            smem_u32(dst)),
        "l"(map), "r"(c0), "r"(c1), "r"(c2), "r"(c3), "r"(smem_u32(bar)), "l"(pol)
        : "memory");
}

// VR = true (static reference state, v1 = v): the velocity tiles are not converted at all -- they land in a 5-slot ring of
// their own and the stencils read them where TMA put them (planes j .. j+4 are alive: the centre plane, the two that
// wait for their turn, the one being converted and the one in flight); raw and sring hold the other fields only.
template <int TZ, int NRAW, int NF, bool VR>
struct RhsTmaSmem {
    static constexpr int HT = (TZ + 4) * SW;
    static constexpr int NH = 4 * TR + 4 * TZ;
    static constexpr int HTP = (HT + 15) / 16 * 16;   // every TMA destination 128-byte aligned
    static constexpr int NFR = VR ? NF - 3 : NF;      // fields per raw buffer
    static constexpr int NV = VR ? NRAW + 3 : 1;      // slots of the velocity ring: planes j .. j+2 in use + NRAW in flight
    static constexpr int NS = VR ? 2 : 5;             // fields of sring
    // TMA destinations of one plane, tile with halo.  VR: rho, p, B (3), J1 (3) [, G (3)]; else U (8), J1 (3) [, G (3)]
    alignas(128) double raw[NRAW][NFR][HTP];
    alignas(128) double vring[NV][3][HTP];            // VR: v_R, v_phi, v_Z of planes n % 5 (TMA destinations)
    // 4-slot rings, tile with halo, written once when a plane arrives (as plane j+2) and read by the in-plane
    // stencils when it is the centre plane (two iterations later).  Four slots, not three: the slot that receives
    // plane j+2 held plane j-2, whose last readers are separated from this write by the barrier of iteration j-1.
    double sring[4][NS][HT];           // rho1, p1 (, v1)
    double ering[4][3][HT];            // E1
    alignas(8) unsigned long long bar[NRAW];   // TMA completion, one per raw buffer
    alignas(8) unsigned long long ready;       // split CTA barrier: "this plane is staged" (one arrival per warp)
};

// the velocity ring is used with a static reference state and the finite-difference phi scheme (with the pre-pass
// derivatives of the pseudo-spectral scheme it measured 4-6 % slower than converting v like the other fields)
__host__ __device__ constexpr bool rhs_velocity_ring(bool v0, bool spec) { return !v0 && !spec; }

// SLAB = true: the context is a slab of a larger grid (owned rows set and / or neighbours linked): a stage writes the
// owned rows only and stores the rows a linked neighbour needs into its ghost rows too.  A separate instantiation, so that
// the undivided path pays nothing for it (measured: +2.3 % on the step when the row tests sit in the default kernel).
template <int TZ, int NRAW, int MODE, bool V0, bool HALL, bool SPEC, bool SLAB>
__global__ void __launch_bounds__(TR *TZ, 1)
rhs_tma_kernel(const __grid_constant__ RhsArgs a, const __grid_constant__ CUtensorMap tmU, const __grid_constant__ CUtensorMap tmJ,
               const __grid_constant__ CUtensorMap tmV)
{
    // tmU: box over the field axis of the stage state -- all 8 fields (moving reference state) or 2 (rho, p; VR);
    // tmV: box of 3 fields (VR: v at field 2, B at field 5); tmJ: J1 [and G]
    extern __shared__ __align__(128) unsigned char smem_raw[];
    constexpr int NF = HALL ? 14 : 11;
    constexpr bool VR = rhs_velocity_ring(V0, SPEC);
    using SM = RhsTmaSmem<TZ, NRAW, NF, VR>;
    SM &S = *reinterpret_cast<SM *>(smem_raw);
    constexpr int HT = SM::HT, NH = SM::NH;
    constexpr int IB = VR ? 2 : 5, IJ = VR ? 5 : 8;      // where B and J1 sit in a raw buffer
    static_assert(NH <= TR * TZ, "tile too small for one halo node per thread");
    const Layout &L = a.L;
    const Phys &ph = a.ph;

    const int tx = threadIdx.x, ty = threadIdx.y, tid = ty * TR + tx;
    const int i0 = 2 + TR * blockIdx.x, k0 = 2 + TZ * blockIdx.y;
    const int i = i0 + tx, k = k0 + ty;
    // a slab's stage writes the context's owned rows only (clt_rhs: every interior row)
    const bool valid = (i <= L.nR - 3) && (k <= L.nZ - 3) && (!SLAB || MODE == RHS_MODE_K || (k >= a.own_k0 && k <= a.own_k1));
    const int ic = min(i, L.nR - 1), kc = min(k, L.nZ - 1);
    const int ja = (int)(((long long)L.nphi * blockIdx.z) / a.phi_chunks);
    const int jb = (int)(((long long)L.nphi * (blockIdx.z + 1)) / a.phi_chunks);
    const long long off2 = (long long)kc * L.pR + (LP + ic);
    const int cs = (ty + 2) * SW + (tx + 2);

    // halo nodes: 4 full rows (Z halo) then 4 columns (R halo), NH in all; the first NH threads take one each (dealing
    // them out evenly over the warps was measured 3 % slower: every warp then pays the divergent halo path)
    const bool is_halo = tid < NH;
    int hx, hy;
    if (tid < 4 * TR) {
        const int r = tid / TR;
        hx = tid % TR;
        hy = (r < 2) ? r - 2 : TZ + (r - 2);
    } else {
        const int t = tid - 4 * TR, c = t & 3;
        hy = t >> 2;
        hx = (c < 2) ? c - 2 : TR + (c - 2);
    }
    const int hi = min(i0 + hx, L.nR - 1), hk = min(k0 + hy, L.nZ - 1);
    const long long hoff2 = (long long)hk * L.pR + (LP + hi);
    const int hs = (hy + 2) * SW + (hx + 2);

    if (tid == 0) {
        for (int b = 0; b < NRAW; ++b) mbar_init(&S.bar[b], 1);
        mbar_init(&S.ready, TZ);         // one arrival per warp (lane 0, after __syncwarp)
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
        asm volatile("prefetch.tensormap [%0];" ::"l"(&tmU) : "memory");
        asm volatile("prefetch.tensormap [%0];" ::"l"(&tmJ) : "memory");
        if (VR) asm volatile("prefetch.tensormap [%0];" ::"l"(&tmV) : "memory");
    }
    __syncthreads();

    const double *tab = a.tab;
    const double eta = ph.eta;
    // planes are numbered n = 0, 1, .. from ja-2; plane n uses raw buffer n % NRAW, its (n / NRAW)-th use
    int nlead = 0;     // number of the plane the next lead() consumes

    // one elected thread: fetch the 11 fields of plane number n (tile with halo) into its raw buffer
    auto issue = [&](int n) {
        const int jw = wrap_phi(ja - 2 + n, L.nphi);
        const int b = n % NRAW;
        mbar_expect_tx(&S.bar[b], (unsigned)(NF * HT * sizeof(double)));
        // two (VR: four) bulk copies per plane: the boxes span the field axis (fields of U; J1 [and G]), so the one thread that
        // issues them -- and the warp that waits for it at the next barrier -- loses a dozen instructions, not a hundred
        static_assert(SM::HTP == HT, "a box that spans the field axis fills the raw buffer densely");
        tma_load_4d(&S.raw[b][0][0], &tmU, LP + i0 - 2, k0 - 2, jw, 0, &S.bar[b]);
        if (VR) {
            tma_load_4d(&S.vring[n % SM::NV][0][0], &tmV, LP + i0 - 2, k0 - 2, jw, 2, &S.bar[b]);
            tma_load_4d(&S.raw[b][IB][0], &tmV, LP + i0 - 2, k0 - 2, jw, 5, &S.bar[b]);
        }
        tma_load_4d(&S.raw[b][IJ][0], &tmJ, LP + i0 - 2, k0 - 2, jw, 0, &S.bar[b]);
    };

    // NRAW planes are kept in flight; the first ones are requested before anything else so that the table reads below
    // overlap their latency
    const int total = jb - ja + 4;
    if (tid == 0)
        for (int n = 0; n < NRAW && n < total; ++n) issue(n);

    // phi-invariant values of the own node and of the halo node, kept in registers for the whole sweep
    const CentreTab ct = load_centre_tab(tab, L.plane, off2);
    const double b0R = __ldg(tab + T_B0R * L.plane + off2), b0P = __ldg(tab + T_B0P * L.plane + off2),
                 b0Z = __ldg(tab + T_B0Z * L.plane + off2);
    const double j0R = __ldg(tab + T_J0R * L.plane + off2), j0P = __ldg(tab + T_J0P * L.plane + off2),
                 j0Z = __ldg(tab + T_J0Z * L.plane + off2);
    const double h_rho0 = __ldg(tab + T_RHO0 * L.plane + hoff2), h_p0 = __ldg(tab + T_P0 * L.plane + hoff2);
    const double rr[4] = { __ldg(a.R + min(i - 2, L.nR - 1)), __ldg(a.R + min(i - 1, L.nR - 1)), __ldg(a.R + min(i + 1, L.nR - 1)),
                           __ldg(a.R + min(i + 2, L.nR - 1)) };

    // forms perturbations, E1 and (optionally) F from the raw tile at slot s; o2 = table offset of the node
    auto node = [&](const double (*raw)[SM::HTP], const double (*vel)[SM::HTP], int s, long long o2, double rho0, double p0,
                    double q[5], double E[3], double F[3], bool wantF) {
        const double rho = raw[0][s], p = raw[1][s];
        const double vR = vel[0][s], vP = vel[1][s], vZ = vel[2][s];
        const double BR = raw[IB][s], BP = raw[IB + 1][s], BZ = raw[IB + 2][s];
        const double JR = raw[IJ][s], JP = raw[IJ + 1][s], JZ = raw[IJ + 2][s];
        q[0] = rho - rho0;
        q[1] = p - p0;
        if (V0) {
            q[2] = vR - __ldg(tab + T_V0R * L.plane + o2);
            q[3] = vP - __ldg(tab + T_V0P * L.plane + o2);
            q[4] = vZ - __ldg(tab + T_V0Z * L.plane + o2);
        } else {
            q[2] = vR; q[3] = vP; q[4] = vZ;
        }
        // a4: E1 = -v x B + v0 x B0 + eta J1   (eq 5 with d_i = 0 minus E0, L77, L101)
        E[0] = eta * JR - (vP * BZ - vZ * BP);
        E[1] = eta * JP - (vZ * BR - vR * BZ);
        E[2] = eta * JZ - (vR * BP - vP * BR);
        if (V0) {
            E[0] += __ldg(tab + T_E0R * L.plane + o2);
            E[1] += __ldg(tab + T_E0P * L.plane + o2);
            E[2] += __ldg(tab + T_E0Z * L.plane + o2);
        }
        if (HALL) {      // Hall term of eq (5): + d_i G (reading R11); G = 0 on the boundary layers
            E[0] = fma(ph.d_i, raw[IJ + 3][s], E[0]);
            E[1] = fma(ph.d_i, raw[IJ + 4][s], E[1]);
            E[2] = fma(ph.d_i, raw[IJ + 5][s], E[2]);
        }
        if (wantF) {
            const double B1R = BR - b0R, B1P = BP - b0P, B1Z = BZ - b0Z;
            F[0] = (JP * BZ - JZ * BP) + (j0P * B1Z - j0Z * B1P);
            F[1] = (JZ * BR - JR * BZ) + (j0Z * B1R - j0R * B1Z);
            F[2] = (JR * BP - JP * BR) + (j0R * B1P - j0P * B1R);
        }
    };

    // thread-private phi pipelines at the own node (slot 4 = newest plane; shifted once per plane)
    double q[5][5];        // rho1, p1, v1 of planes j-2 .. j+2
    double eR[5], eZ[5];   // E1_R, E1_Z of planes j-2 .. j+2
    double Fp[3][3];       // F = J1 x B + J0 x B1 of planes j .. j+2
    int sl = 0;            // ring slot that receives the plane being consumed (plane j+2)

    // consume the raw tile of plane number nlead (the plane that becomes plane j+2)
    auto lead = [&]() {
        const int b = nlead % NRAW;
        mbar_wait(&S.bar[b], (unsigned)((nlead / NRAW) & 1));
        const double (*raw)[SM::HTP] = S.raw[b];
        const double (*vel)[SM::HTP] = VR ? S.vring[nlead % SM::NV] : S.raw[b] + 2;
        ++nlead;
        double E[3];
        node(raw, vel, cs, off2, ct.rho0, ct.p0, q[4], E, Fp[2], true);
        eR[4] = E[0];
        eZ[4] = E[2];
#pragma unroll
        for (int c = 0; c < 3; ++c) S.ering[sl][c][cs] = E[c];
#pragma unroll
        for (int f = 0; f < SM::NS; ++f) S.sring[sl][f][cs] = q[4][f];
        if (is_halo) {
            double hq[5], hE[3], hF[3];
            node(raw, vel, hs, hoff2, h_rho0, h_p0, hq, hE, hF, false);
#pragma unroll
            for (int c = 0; c < 3; ++c) S.ering[sl][c][hs] = hE[c];
#pragma unroll
            for (int f = 0; f < SM::NS; ++f) S.sring[sl][f][hs] = hq[f];
        }
    };
    auto advance = [&]() {
#pragma unroll
        for (int d = 0; d < 4; ++d) {
#pragma unroll
            for (int f = 0; f < 5; ++f) q[d][f] = q[d + 1][f];
            eR[d] = eR[d + 1];
            eZ[d] = eZ[d + 1];
        }
#pragma unroll
        for (int c = 0; c < 3; ++c) { Fp[0][c] = Fp[1][c]; Fp[1][c] = Fp[2][c]; }
        sl = (sl + 1) & 3;
    };

    // prologue: planes number 0 .. 3 (ja-2 .. ja+1)
#pragma unroll 1
    for (int n = 0; n < 4; ++n) {
        lead();
        __syncthreads();                 // every thread has read the raw tile
        if (tid == 0 && n + NRAW < total) issue(n + NRAW);
        advance();
    }

    const double iR = __ldg(a.invR + ic);
    const double iR2 = iR * iR;
    double rate = 0.0;           // largest signal rate (|v_d| + c)/(12 h_d) at this thread's nodes (stage 4 of clt_step_cfl)
    const StageCoef coef = load_stage_coef<MODE>(a);

#pragma unroll 1
    for (int j = ja; j < jb; ++j) {
        // ---- phase A: consume plane j+2 --------------------------------------------------------
        if (a.prefetch && MODE != RHS_MODE_K && (tx & 15) == 0 && j + 1 < jb) {
            const long long g1 = (long long)(j + 1) * L.plane + off2;
#pragma unroll
            for (int m = 0; m < 8; ++m) {
                if (MODE != RHS_MODE_S1) prefetch_l2(a.Un + m * L.field + g1);
                if (MODE == RHS_MODE_S4) prefetch_l2(a.acc + m * L.field + g1);
            }
        }
        const int it = j - ja;                                    // iteration number: consumes plane number it + 4
        lead();
        const int sc = (sl + 2) & 3;                              // ring slot of the centre plane
        // split barrier: announce "my part of plane j+2 is in the rings", keep working on what needs nobody else's
        // data (epilogue operand loads, the phi direction), and only then wait for the other warps
        __syncwarp();
        if (tx == 0) mbar_arrive(&S.ready);

        // ---- a6 inputs: U^n / stage state / acc of this node, requested now so that they arrive during phase B ---
        const long long g = (long long)j * L.plane + off2;
        EpiOperands eo;
        // rho, p (and v when the reference state is static) of the centre plane are still in the phi pipeline
        constexpr int NOWN = V0 ? 2 : 5;
        const double own[5] = { q[2][0] + ct.rho0, q[2][1] + ct.p0, q[2][2], q[2][3], q[2][4] };
        epilogue_load<MODE, NOWN>(a, g, L.field, eo, [](const double *p) { return ld_stream(p); }, own);

        // ---- phase B: K at (i, k, j) -----------------------------------------------------------
        double K[8];
        double dP_EZ, dP_ER, pd1[5], pd2[5];
        if (SPEC) {
            // pseudo-spectral phi derivatives of this node from the pre-pass (requested with the epilogue operands)
#pragma unroll
            for (int f = 0; f < 5; ++f) {
                pd1[f] = ld_stream(a.spec + (SP_D1 + f) * L.field + g);
                pd2[f] = ld_stream(a.spec + (SP_D2 + f) * L.field + g);
            }
            dP_ER = ld_stream(a.spec + (SP_DE + 0) * L.field + g);
            dP_EZ = ld_stream(a.spec + (SP_DE + 1) * L.field + g);
        } else {
            dP_EZ = fd1(eZ[0], eZ[1], eZ[3], eZ[4]);
            dP_ER = fd1(eR[0], eR[1], eR[3], eR[4]);
        }
        // velocity tiles of the centre plane (plane number it + 2): as they arrived (VR), or converted (sring fields 2-4)
        const double *velc = VR ? &S.vring[(it + 2) % SM::NV][0][0] : &S.sring[sc][SM::NS - 3][0];
        rhs_point<V0, SPEC>(&S.sring[sc][0][0], velc, HT, &S.ering[sc][0][0], &S.ering[sc][1][0], &S.ering[sc][2][0], dP_EZ, dP_ER, Fp[0],
                            rr, cs, q, ct, tab, off2, L.plane, ph, iR, iR2, K, [&] {
                                mbar_wait(&S.ready, (unsigned)(it & 1));
                                // every thread has consumed the raw buffer of plane number it+4: refill it NRAW planes
                                // ahead (overlaps the rest of phase B and NRAW-1 more iterations)
                                const int n = it + 4 + NRAW;
                                if (tid == 0 && n < total) issue(n);
                            }, pd1, pd2);

        // ---- a6: RK4 stage combine in the epilogue (L125, L139) --------------------------------
        if (valid) {
            if (SLAB)
                epilogue_store<MODE>(a, g, L.field, eo, K, iR, rate, coef, true, peer_node(a, 0, i, k, j, L.pR), peer_node(a, 1, i, k, j, L.pR));
            else
                epilogue_store<MODE>(a, g, L.field, eo, K, iR, rate, coef, true);
        }
        advance();
    }
    if (MODE == RHS_MODE_S4) dtmin_commit(a, rate);
}

template <int MODE, bool V0, bool HALL, bool SPEC, bool SLAB>
static cudaError_t launch_rhs_tma_t(const RhsArgs &a, const CUtensorMap &tmU, const CUtensorMap &tmJ, const CUtensorMap &tmV,
                                    cudaStream_t s, bool configure)
{
    // raw buffers (planes in flight): two; three in stage 1 where the shared memory is there (velocity ring, no Hall
    // field).  Measured at 512x64x512: stage 1 (latency-bound, its prologue waits for every plane) 0.555 -> 0.540 ms with
    // three, the HBM-bound stages 2 and 4 +2 % and +4 % slower, stage 3 unchanged.
    constexpr int TZ = RHS_TZ, NRAW = (MODE == RHS_MODE_S1 && rhs_velocity_ring(V0, SPEC) && !HALL) ? 3 : 2;
    auto kern = rhs_tma_kernel<TZ, NRAW, MODE, V0, HALL, SPEC, SLAB>;
    using SM = RhsTmaSmem<TZ, NRAW, HALL ? 14 : 11, rhs_velocity_ring(V0, SPEC)>;
    const int smem = (int)sizeof(SM);
    static_assert(sizeof(SM) <= 232448, "shared memory of the TMA RHS kernel exceeds 227 KB");
    if (configure) return cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, smem);
    dim3 block(TR, TZ, 1);
    dim3 grid((a.L.nR - 4 + TR - 1) / TR, (a.L.nZ - 4 + TZ - 1) / TZ, a.phi_chunks);
    kern<<<grid, block, smem, s>>>(a, tmU, tmJ, tmV);
    return cudaGetLastError();
}

template <bool HALL, bool SPEC>
static cudaError_t launch_rhs_tma_hs(const RhsArgs &a, const CUtensorMap &tmU, const CUtensorMap &tmJ, const CUtensorMap &tmV, int mode,
                                     bool v0, bool slab, cudaStream_t s, bool configure)
{
    // clt_rhs (mode K) has no slab variant: it writes every interior row of a scratch buffer
    if (mode == RHS_MODE_K)
        return v0 ? launch_rhs_tma_t<RHS_MODE_K, true, HALL, SPEC, false>(a, tmU, tmJ, tmV, s, configure)
                  : launch_rhs_tma_t<RHS_MODE_K, false, HALL, SPEC, false>(a, tmU, tmJ, tmV, s, configure);
#define CLT_CASE(M)                                                                                                         \
    case M:                                                                                                                 \
        if (slab)                                                                                                           \
            return v0 ? launch_rhs_tma_t<M, true, HALL, SPEC, true>(a, tmU, tmJ, tmV, s, configure)                         \
                      : launch_rhs_tma_t<M, false, HALL, SPEC, true>(a, tmU, tmJ, tmV, s, configure);                       \
        return v0 ? launch_rhs_tma_t<M, true, HALL, SPEC, false>(a, tmU, tmJ, tmV, s, configure)                            \
                  : launch_rhs_tma_t<M, false, HALL, SPEC, false>(a, tmU, tmJ, tmV, s, configure);
    switch (mode) {
        CLT_CASE(RHS_MODE_S1)
        CLT_CASE(RHS_MODE_S2)
        CLT_CASE(RHS_MODE_S3)
        CLT_CASE(RHS_MODE_S4)
    default:
        return cudaErrorInvalidValue;
    }
#undef CLT_CASE
}

cudaError_t launch_rhs_tma(const RhsArgs &a, const void *tmU, const void *tmJ, const void *tmV, int mode, bool has_v0, bool hall,
                           bool spec, bool slab, cudaStream_t s, bool configure)
{
    const CUtensorMap &mU = *reinterpret_cast<const CUtensorMap *>(tmU);
    const CUtensorMap &mJ = *reinterpret_cast<const CUtensorMap *>(tmJ);
    const CUtensorMap &mV = *reinterpret_cast<const CUtensorMap *>(tmV);
    if (hall && spec) return launch_rhs_tma_hs<true, true>(a, mU, mJ, mV, mode, has_v0, slab, s, configure);
    if (hall) return launch_rhs_tma_hs<true, false>(a, mU, mJ, mV, mode, has_v0, slab, s, configure);
    if (spec) return launch_rhs_tma_hs<false, true>(a, mU, mJ, mV, mode, has_v0, slab, s, configure);
    return launch_rhs_tma_hs<false, false>(a, mU, mJ, mV, mode, has_v0, slab, s, configure);
}

// ---------------------------------------------------------------------------------------------
// curl_kernel: J1 = curl_c(B - B0) on interior nodes (eq 6).  Same sweep, 3 staged fields.
// ---------------------------------------------------------------------------------------------
template <int TZ>
struct CurlSmem {
    static constexpr int HT = (TZ + 4) * SW;
    double stage[2][3][HT];    // B1_R, B1_phi, B1_Z of the centre plane
    double sR[SW];
};

template <int TZ>
__global__ void __launch_bounds__(TR *TZ, 2) curl_kernel(const __grid_constant__ CurlArgs a)
{
    __shared__ CurlSmem<TZ> S;
    const Layout &L = a.L;
    const Phys &ph = a.ph;
    const int tx = threadIdx.x, ty = threadIdx.y, tid = ty * TR + tx;
    const int i0 = 2 + TR * blockIdx.x, k0 = 2 + TZ * blockIdx.y;
    const int i = i0 + tx, k = k0 + ty;
    const bool valid = (i <= L.nR - 3) && (k <= L.nZ - 3);
    const int ic = min(i, L.nR - 1), kc = min(k, L.nZ - 1);
    const int ja = (int)(((long long)L.nphi * blockIdx.z) / a.phi_chunks);
    const int jb = (int)(((long long)L.nphi * (blockIdx.z + 1)) / a.phi_chunks);
    const long long off2 = (long long)kc * L.pR + (LP + ic);
    const int cs = (ty + 2) * SW + (tx + 2);

    constexpr int NH = 4 * TR + 4 * TZ;
    static_assert(NH <= TR * TZ, "tile too small for one halo node per thread");
    int hx, hy;
    if (tid < 4 * TR) {
        const int r = tid / TR;
        hx = tid % TR;
        hy = (r < 2) ? r - 2 : TZ + (r - 2);
    } else {
        const int t = tid - 4 * TR, c = t & 3;
        hy = t >> 2;
        hx = (c < 2) ? c - 2 : TR + (c - 2);
    }
    const bool is_halo = tid < NH;
    const int hi = min(i0 + hx, L.nR - 1), hk = min(k0 + hy, L.nZ - 1);
    const long long hoff2 = (long long)hk * L.pR + (LP + hi);
    const int hs = (hy + 2) * SW + (hx + 2);
    if (tid < SW) S.sR[tid] = a.R[min(i0 - 2 + tid, L.nR - 1)];

    const double *tab = a.tab;
    const double b0R = __ldg(tab + T_B0R * L.plane + off2), b0P = __ldg(tab + T_B0P * L.plane + off2),
                 b0Z = __ldg(tab + T_B0Z * L.plane + off2);
    double h0R = 0.0, h0P = 0.0, h0Z = 0.0;
    if (is_halo) {
        h0R = __ldg(tab + T_B0R * L.plane + hoff2);
        h0P = __ldg(tab + T_B0P * L.plane + hoff2);
        h0Z = __ldg(tab + T_B0Z * L.plane + hoff2);
    }
    const double iR = __ldg(a.invR + ic);

    double bR[5], bZ[5], bP[3];    // B1 of planes j-2..j+2 (R, Z) and j..j+2 (phi) at the own node
    auto lead = [&](int jl) {
        const long long g = (long long)wrap_phi(jl, L.nphi) * L.plane + off2;
        bR[4] = __ldg(a.B + 0 * L.field + g) - b0R;    // equilibrium subtracted before differencing (H2)
        bP[2] = __ldg(a.B + 1 * L.field + g) - b0P;
        bZ[4] = __ldg(a.B + 2 * L.field + g) - b0Z;
    };
    auto advance = [&]() {
#pragma unroll
        for (int d = 0; d < 4; ++d) { bR[d] = bR[d + 1]; bZ[d] = bZ[d + 1]; }
        bP[0] = bP[1]; bP[1] = bP[2];
    };
#pragma unroll 1
    for (int jl = ja - 2; jl <= ja + 1; ++jl) { lead(jl); advance(); }

#pragma unroll 1
    for (int j = ja; j < jb; ++j) {
        const int buf = j & 1;
        lead(j + 2);
        S.stage[buf][0][cs] = bR[2];
        S.stage[buf][1][cs] = bP[0];
        S.stage[buf][2][cs] = bZ[2];
        if (is_halo) {
            const long long g = (long long)j * L.plane + hoff2;
            S.stage[buf][0][hs] = __ldg(a.B + 0 * L.field + g) - h0R;
            S.stage[buf][1][hs] = __ldg(a.B + 1 * L.field + g) - h0P;
            S.stage[buf][2][hs] = __ldg(a.B + 2 * L.field + g) - h0Z;
        }
        __syncthreads();
        const double *sBR = &S.stage[buf][0][cs], *sBP = &S.stage[buf][1][cs], *sBZ = &S.stage[buf][2][cs];
        const double cPi = ph.cP1 * iR;
        const double dP_BZ = fd1(bZ[0], bZ[1], bZ[3], bZ[4]);
        const double dP_BR = fd1(bR[0], bR[1], bR[3], bR[4]);
        const double dZ_BP = fd1(sBP[-2 * SW], sBP[-SW], sBP[SW], sBP[2 * SW]);
        const double dZ_BR = fd1(sBR[-2 * SW], sBR[-SW], sBR[SW], sBR[2 * SW]);
        const double dR_BZ = fd1(sBZ[-2], sBZ[-1], sBZ[1], sBZ[2]);
        const double *r = &S.sR[tx + 2];
        const double dR_RBP = fd1(r[-2] * sBP[-2], r[-1] * sBP[-1], r[1] * sBP[1], r[2] * sBP[2]);
        if (valid) {
            const long long g = (long long)j * L.plane + off2;
            a.J1[0 * L.field + g] = dP_BZ * cPi - dZ_BP * ph.cZ1;
            a.J1[1 * L.field + g] = dZ_BR * ph.cZ1 - dR_BZ * ph.cR1;
            a.J1[2 * L.field + g] = dR_RBP * (ph.cR1 * iR) - dP_BR * cPi;
        }
        advance();
    }
}

cudaError_t launch_curl(const CurlArgs &a, cudaStream_t s)
{
    constexpr int TZ = 8;
    dim3 block(TR, TZ, 1);
    dim3 grid((a.L.nR - 4 + TR - 1) / TR, (a.L.nZ - 4 + TZ - 1) / TZ, a.phi_chunks);
    curl_kernel<TZ><<<grid, block, 0, s>>>(a);
    return cudaGetLastError();
}

// ---------------------------------------------------------------------------------------------
// TMA variant of the curl kernel (the default): an NS-deep shared-memory ring of raw B tiles (with
// halo) filled by cp.async.bulk.tensor three planes ahead; threads read their stencil neighbours
// straight from the ring and subtract the (phi-invariant) B0 values they keep in registers, so the
// equilibrium is still removed before differencing (H2).  No staging, one __syncthreads per plane
// (only to hand the consumed ring slot back to the producer thread).
// ---------------------------------------------------------------------------------------------
template <int TZ, int NS, int NF>
struct CurlTmaSmem {
    static constexpr int HT = (TZ + 4) * SW;
    static constexpr int HTP = (HT + 15) / 16 * 16;
    alignas(128) double raw[NS][NF][HTP];      // B_R, B_phi, B_Z (and rho, p for the Hall variant)
    alignas(8) unsigned long long full[NS];
};

// HALL = true additionally forms the Hall field of eq (5) [L77] in its equilibrium-subtracted form (DESIGN.md
// reading R11),  G = (J1 x B + J0 x B1 - grad p1)/rho - (rho1/rho)(v0.grad)v0,  on interior nodes: the same sweep
// with rho and p staged next to B (p1 = p - p0 is formed before differencing, H2).  tmU maps the whole stage state.
// SPEC = true takes d/dphi of B1_R, B1_Z (and p1) from the pseudo-spectral pre-pass instead of the phi stencil.
template <int TZ, int NS, bool HALL, bool SPEC>
__global__ void __launch_bounds__(TR *TZ, HALL ? 1 : CLT_CURL_MINB)
curl_tma_kernel(const __grid_constant__ CurlArgs a, const __grid_constant__ CUtensorMap tmU)
{
    extern __shared__ __align__(128) unsigned char smem_raw[];
    constexpr int NF = HALL ? 5 : 3;
    using SM = CurlTmaSmem<TZ, NS, NF>;
    SM &S = *reinterpret_cast<SM *>(smem_raw);
    const Layout &L = a.L;
    const Phys &ph = a.ph;
    const int tx = threadIdx.x, ty = threadIdx.y, tid = ty * TR + tx;
    const int i0 = 2 + TR * blockIdx.x, k0 = 2 + TZ * blockIdx.y;
    const int i = i0 + tx, k = k0 + ty;
    const bool valid = (i <= L.nR - 3) && (k <= L.nZ - 3);
    const int ic = min(i, L.nR - 3), kc = min(k, L.nZ - 3);     // clamped to an interior node: +-2 stays in range
    const int ja = (int)(((long long)L.nphi * blockIdx.z) / a.phi_chunks);
    const int jb = (int)(((long long)L.nphi * (blockIdx.z + 1)) / a.phi_chunks);
    const long long off2 = (long long)kc * L.pR + (LP + ic);
    const int cs = (ty + 2) * SW + (tx + 2);
    const int total = jb - ja + 4;                               // planes ja-2 .. jb+1

    if (tid == 0) {
        for (int n = 0; n < NS; ++n) mbar_init(&S.full[n], 1);
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
        asm volatile("prefetch.tensormap [%0];" ::"l"(&tmU) : "memory");
    }
    __syncthreads();
    auto issue = [&](int n) {      // plane number n counts from ja-2
        const int jw = wrap_phi(ja - 2 + n, L.nphi);
        const int st = n % NS;
        mbar_expect_tx(&S.full[st], (unsigned)(NF * SM::HT * sizeof(double)));
#pragma unroll
        for (int m = 0; m < 3; ++m) tma_load_4d(&S.raw[st][m][0], &tmU, LP + i0 - 2, k0 - 2, jw, 5 + m, &S.full[st]);
        if (HALL) {
            tma_load_4d(&S.raw[st][3][0], &tmU, LP + i0 - 2, k0 - 2, jw, 0, &S.full[st]);
            tma_load_4d(&S.raw[st][4][0], &tmU, LP + i0 - 2, k0 - 2, jw, 1, &S.full[st]);
        }
    };
    if (tid == 0)
        for (int n = 0; n < NS && n < total; ++n) issue(n);

    // phi-invariant operands in registers: B0 at the own node and at the 8 in-plane neighbours, R_i
    const double *tab = a.tab;
    const double *t0R = tab + T_B0R * L.plane + off2, *t0P = tab + T_B0P * L.plane + off2, *t0Z = tab + T_B0Z * L.plane + off2;
    const double o0R = __ldg(t0R), o0Z = __ldg(t0Z);
    double z0P[4], z0R[4], r0Z[4], r0P[4], rr[4];
    double zp0[4], rp0[4];          // p0 at the in-plane neighbours (Hall)
#pragma unroll
    for (int d = 0; d < 4; ++d) {
        const int o = (d < 2) ? d - 2 : d - 1;          // -2, -1, +1, +2
        z0P[d] = __ldg(t0P + (long long)o * L.pR);
        z0R[d] = __ldg(t0R + (long long)o * L.pR);
        r0Z[d] = __ldg(t0Z + o);
        r0P[d] = __ldg(t0P + o);
        rr[d] = __ldg(a.R + ic + o);
        if (HALL) {
            zp0[d] = __ldg(tab + T_P0 * L.plane + off2 + (long long)o * L.pR);
            rp0[d] = __ldg(tab + T_P0 * L.plane + off2 + o);
        }
    }
    double o0P = 0.0, rho0 = 0.0, j0R = 0.0, j0P = 0.0, j0Z = 0.0, a0R = 0.0, a0P = 0.0, a0Z = 0.0;
    if (HALL) {
        o0P = __ldg(t0P);
        rho0 = __ldg(tab + T_RHO0 * L.plane + off2);
        j0R = __ldg(tab + T_J0R * L.plane + off2); j0P = __ldg(tab + T_J0P * L.plane + off2); j0Z = __ldg(tab + T_J0Z * L.plane + off2);
        a0R = __ldg(tab + T_A0R * L.plane + off2); a0P = __ldg(tab + T_A0P * L.plane + off2); a0Z = __ldg(tab + T_A0Z * L.plane + off2);
    }
    const double iR = __ldg(a.invR + ic);
    const double cPi = ph.cP1 * iR;

    double bR[5], bZ[5];           // B1_R, B1_Z of planes j-2 .. j+2 at the own node
    double pP[5];                  // p of planes j-2 .. j+2 at the own node (Hall; d_phi p1 = d_phi p)
    auto lead = [&](int n) {
        const int st = n % NS;
        mbar_wait(&S.full[st], (unsigned)((n / NS) & 1));
        bR[4] = S.raw[st][0][cs] - o0R;
        bZ[4] = S.raw[st][2][cs] - o0Z;
        if (HALL) pP[4] = S.raw[st][NF - 1][cs];
    };
    auto advance = [&]() {
#pragma unroll
        for (int d = 0; d < 4; ++d) {
            bR[d] = bR[d + 1];
            bZ[d] = bZ[d + 1];
            if (HALL) pP[d] = pP[d + 1];
        }
    };
#pragma unroll 1
    for (int n = 0; n < 4; ++n) { lead(n); advance(); }
    __syncthreads();                                   // planes 0 and 1 are never centre planes: recycle their slots
    if (tid == 0) {
        if (NS < total) issue(NS);
        if (NS + 1 < total) issue(NS + 1);
    }

#pragma unroll 1
    for (int j = ja; j < jb; ++j) {
        const int nc = j - ja + 2;                     // plane number of the centre plane
        lead(nc + 2);
        const int st = nc % NS;
        const double *sR_ = &S.raw[st][0][cs], *sP_ = &S.raw[st][1][cs], *sZ_ = &S.raw[st][2][cs];
        const double dP_BZ = fd1(bZ[0], bZ[1], bZ[3], bZ[4]);
        const double dP_BR = fd1(bR[0], bR[1], bR[3], bR[4]);
        const double dZ_BP = fd1(sP_[-2 * SW] - z0P[0], sP_[-SW] - z0P[1], sP_[SW] - z0P[2], sP_[2 * SW] - z0P[3]);
        const double dZ_BR = fd1(sR_[-2 * SW] - z0R[0], sR_[-SW] - z0R[1], sR_[SW] - z0R[2], sR_[2 * SW] - z0R[3]);
        const double dR_BZ = fd1(sZ_[-2] - r0Z[0], sZ_[-1] - r0Z[1], sZ_[1] - r0Z[2], sZ_[2] - r0Z[3]);
        const double dR_RBP = fd1(rr[0] * (sP_[-2] - r0P[0]), rr[1] * (sP_[-1] - r0P[1]), rr[2] * (sP_[1] - r0P[2]),
                                  rr[3] * (sP_[2] - r0P[3]));
        const long long gc = (long long)j * L.plane + off2;
        const double pBZ = SPEC ? __ldg(a.spec + (SP_DB + 1) * L.field + gc) * iR : dP_BZ * cPi;     // d_phi B1_Z / R
        const double pBR = SPEC ? __ldg(a.spec + (SP_DB + 0) * L.field + gc) * iR : dP_BR * cPi;     // d_phi B1_R / R
        const double JR = pBZ - dZ_BP * ph.cZ1;
        const double JP = dZ_BR * ph.cZ1 - dR_BZ * ph.cR1;
        const double JZ = dR_RBP * (ph.cR1 * iR) - pBR;
        double GR = 0.0, GP = 0.0, GZ = 0.0;
        if (HALL) {
            const double *sp_ = &S.raw[st][NF - 1][cs];
            const double rho = S.raw[st][NF - 2][cs];
            const double BR = sR_[0], BP = sP_[0], BZ = sZ_[0];
            const double B1R = bR[2], B1P = BP - o0P, B1Z = bZ[2];
            const double gR = fd1(sp_[-2] - rp0[0], sp_[-1] - rp0[1], sp_[1] - rp0[2], sp_[2] - rp0[3]) * ph.cR1;
            const double gZ = fd1(sp_[-2 * SW] - zp0[0], sp_[-SW] - zp0[1], sp_[SW] - zp0[2], sp_[2 * SW] - zp0[3]) * ph.cZ1;
            const double gP = SPEC ? __ldg(a.spec + (SP_D1 + 1) * L.field + gc) * iR : fd1(pP[0], pP[1], pP[3], pP[4]) * cPi;
            const double rinv = 1.0 / rho, r1 = (rho - rho0) * rinv;
            GR = ((JP * BZ - JZ * BP) + (j0P * B1Z - j0Z * B1P) - gR) * rinv - r1 * a0R;
            GP = ((JZ * BR - JR * BZ) + (j0Z * B1R - j0R * B1Z) - gP) * rinv - r1 * a0P;
            GZ = ((JR * BP - JP * BR) + (j0R * B1P - j0P * B1R) - gZ) * rinv - r1 * a0Z;
        }
        if (valid) {
            const long long g = (long long)j * L.plane + off2;
            a.J1[0 * L.field + g] = JR;
            a.J1[1 * L.field + g] = JP;
            a.J1[2 * L.field + g] = JZ;
            if (HALL) {
                a.G[0 * L.field + g] = GR;
                a.G[1 * L.field + g] = GP;
                a.G[2 * L.field + g] = GZ;
            }
        }
        advance();
        __syncthreads();                               // the centre plane's slot is free again
        if (tid == 0 && nc + NS < total) issue(nc + NS);
    }
}

template <bool HALL, bool SPEC>
static cudaError_t launch_curl_tma_t(const CurlArgs &a, const void *tmU, cudaStream_t s, bool configure)
{
    constexpr int TZ = CLT_CURL_TZ, NS = CLT_CURL_NS;
    auto kern = curl_tma_kernel<TZ, NS, HALL, SPEC>;
    const int smem = (int)sizeof(CurlTmaSmem<TZ, NS, HALL ? 5 : 3>);
    if (configure) return cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, smem);
    dim3 block(TR, TZ, 1);
    dim3 grid((a.L.nR - 4 + TR - 1) / TR, (a.L.nZ - 4 + TZ - 1) / TZ, a.phi_chunks);
    kern<<<grid, block, smem, s>>>(a, *reinterpret_cast<const CUtensorMap *>(tmU));
    return cudaGetLastError();
}

cudaError_t launch_curl_tma(const CurlArgs &a, const void *tmU, bool hall, bool spec, cudaStream_t s, bool configure)
{
    if (spec) return hall ? launch_curl_tma_t<true, true>(a, tmU, s, configure) : launch_curl_tma_t<false, true>(a, tmU, s, configure);
    return hall ? launch_curl_tma_t<true, false>(a, tmU, s, configure) : launch_curl_tma_t<false, false>(a, tmU, s, configure);
}
int curl_tma_tile_z() { return CLT_CURL_TZ; }

// ---------------------------------------------------------------------------------------------
// NEXT-2: pseudo-spectral phi derivatives ("either 4th order finite difference or
// pseudo-spectrum method can be used" in phi; reading R12).  A phi-global operator does not fit
// the phi-marching sweeps, so the derivatives are formed by a pre-pass and read back by the SPEC variants of
// the curl and fused RHS kernels.  A CTA owns 32 neighbouring (R, Z) lines of one quantity: it stages their
// N = nphi samples in shared memory (coalesced, perturbations formed first, H2) and evaluates the circulant sums
// in their paired form
//   d1_j = sum_{m=1..Q} c1[m] (f_{j+m} - f_{j-m}),   Q = floor((N-1)/2)
//   d2_j = c2[0] f_j + sum_{m=1..Q} c2[m] (f_{j+m} + f_{j-m}) [+ c2[N/2] f_{j+N/2}, N even]
// with the closed-form weights of the Fourier differentiation matrices (clt_api.cu).  A thread forms CLT_SPEC_NQ = 8
// consecutive outputs of one line at a time from two sliding register windows, so every step in m costs two
// shared-memory loads for 16 (32 with second derivatives) FP64 operations: FP64-bound, any N <= 256.
// ---------------------------------------------------------------------------------------------
// Stages the N = nphi samples of the quantity pre-pass job `job` differentiates, for the (R, Z) line at table offset o2,
// into sv[j * pitch + tx] (thread (tx, ty) of TY rows takes planes ty, ty + TY, ..: coalesced along R), and names the
// output fields.  Perturbations are formed first (H2).
__device__ __forceinline__ void spec_stage(const SpecArgs &a, int job, long long o2, double *sv, int pitch, int tx, int ty, int TY,
                                           int &out1, int &out2)
{
    const Layout &L = a.L;
    const int N = L.nphi;
    out2 = -1;
    if (a.mode == 0) {
        // before the curl: B1_R, B1_Z (and p1 for the Hall field)
        const int src = job == 0 ? 5 : (job == 1 ? 7 : 1);
        const int t0 = job == 0 ? T_B0R : (job == 1 ? T_B0Z : T_P0);
        out1 = job < 2 ? SP_DB + job : SP_D1 + 1;
        const double f0 = __ldg(a.tab + t0 * L.plane + o2);
        for (int j = ty; j < N; j += TY) sv[j * pitch + tx] = __ldg(a.U + src * L.field + (long long)j * L.plane + o2) - f0;
    } else if (job < 5) {
        out1 = SP_D1 + job;
        out2 = SP_D2 + job;
        const int t0 = job == 0 ? T_RHO0 : (job == 1 ? T_P0 : T_V0R + (job - 2));
        const double f0 = (job < 2 || a.has_v0) ? __ldg(a.tab + t0 * L.plane + o2) : 0.0;
        for (int j = ty; j < N; j += TY) sv[j * pitch + tx] = __ldg(a.U + job * L.field + (long long)j * L.plane + o2) - f0;
    } else {
        // E1_R (job 5) or E1_Z (job 6) = -(v x B)_c + eta J1_c (+ d_i G_c); the axisymmetric v0 x B0 drops out
        // of the paired differences exactly and is left out
        const int c = job == 5 ? 0 : 2;
        out1 = SP_DE + (job - 5);
        // (v x B)_R = v_phi B_Z - v_Z B_phi ; (v x B)_Z = v_R B_phi - v_phi B_R
        const int ia = c == 0 ? 3 : 2, ib = c == 0 ? 7 : 6, ic2 = c == 0 ? 4 : 3, id = c == 0 ? 6 : 5;
        for (int j = ty; j < N; j += TY) {
            const long long g = (long long)j * L.plane + o2;
            const double va = __ldg(a.U + ia * L.field + g), Bb = __ldg(a.U + ib * L.field + g);
            const double vc = __ldg(a.U + ic2 * L.field + g), Bd = __ldg(a.U + id * L.field + g);
            double e = a.ph.eta * __ldg(a.J1 + c * L.field + g) - (va * Bb - vc * Bd);
            if (a.hall) e = fma(a.ph.d_i, __ldg(a.J1 + (3 + c) * L.field + g), e);
            sv[j * pitch + tx] = e;
        }
    }
}

template <bool WANT2>
__global__ void __launch_bounds__(512) phi_spectral_kernel(const __grid_constant__ SpecArgs a, int job_base)
{
    extern __shared__ __align__(128) unsigned char smem_raw[];
    const Layout &L = a.L;
    const int N = L.nphi;
    double *sv = reinterpret_cast<double *>(smem_raw);        // [N][32] samples
    double *sc1 = sv + (size_t)N * 32, *sc2 = sc1 + N;        // weights
    const int tx = threadIdx.x, ty = threadIdx.y, TY = blockDim.y;
    const int i = 2 + blockIdx.x * 32 + tx, k = 2 + blockIdx.y;
    const bool valid = i <= L.nR - 3;
    const long long o2 = (long long)k * L.pR + (LP + min(i, L.nR - 3));
    const int job = job_base + blockIdx.z;
    int out1, out2;            // output field of the first / second derivative (-1: none)
    spec_stage(a, job, o2, sv, 32, tx, ty, TY, out1, out2);
    for (int m = ty * 32 + tx; m < N; m += TY * 32) {
        sc1[m] = a.ctab[m];
        sc2[m] = a.ctab[SPEC_MAX_NPHI + m];
    }
    __syncthreads();

    const int Q = (N - 1) / 2;
    const bool even = (N & 1) == 0, want2 = WANT2 && out2 >= 0;
    const double *v = sv + tx;
    auto wrap = [N](int x) { x %= N; return x < 0 ? x + N : x; };
    constexpr int NQ = CLT_SPEC_NQ;             // outputs per thread and window width
    for (int j0 = NQ * ty; j0 < N; j0 += NQ * TY) {
        double s1[NQ], s2[NQ], wa[NQ], wb[NQ];  // windows: wa[q] = f_{j0+q+m}, wb[q] = f_{j0+q-m}
#pragma unroll
        for (int q = 0; q < NQ; ++q) {
            s1[q] = 0.0;
            s2[q] = WANT2 ? sc2[0] * v[wrap(j0 + q) * 32] : 0.0;
            wa[q] = v[wrap(j0 + q + 1) * 32];
            wb[q] = v[wrap(j0 + q - 1) * 32];
        }
        int pa = wrap(j0 + NQ + 1), pb = wrap(j0 - 2);
#pragma unroll 4
        for (int m = 1; m <= Q; ++m) {
            const double c1 = sc1[m], c2 = sc2[m];
#pragma unroll
            for (int q = 0; q < NQ; ++q) {
                s1[q] = fma(c1, wa[q] - wb[q], s1[q]);
                if (WANT2) s2[q] = fma(c2, wa[q] + wb[q], s2[q]);
            }
#pragma unroll
            for (int q = 0; q < NQ - 1; ++q) wa[q] = wa[q + 1];
            wa[NQ - 1] = v[pa * 32];
#pragma unroll
            for (int q = NQ - 1; q > 0; --q) wb[q] = wb[q - 1];
            wb[0] = v[pb * 32];
            pa = pa + 1 == N ? 0 : pa + 1;
            pb = pb == 0 ? N - 1 : pb - 1;
        }
        if (WANT2 && even) {
#pragma unroll
            for (int q = 0; q < NQ; ++q) s2[q] = fma(sc2[N / 2], v[wrap(j0 + q + N / 2) * 32], s2[q]);
        }
        if (valid) {
#pragma unroll
            for (int q = 0; q < NQ; ++q)
                if (j0 + q < N) {
                    const long long g = (long long)(j0 + q) * L.plane + o2;
                    a.out[(long long)out1 * L.field + g] = s1[q];
                    if (want2) a.out[(long long)out2 * L.field + g] = s2[q];
                }
        }
    }
}

// ---------------------------------------------------------------------------------------------
// N = nphi = 64: the same derivatives through a register-resident FFT (about 6 x fewer FP64 operations than the circulant
// sums; the pre-pass becomes HBM-bound).  Two neighbouring real lines a, b are packed as z = a + i b: the derivative is
// a real-linear operator, so multiplying the spectrum of z by i kappa q (resp. -(kappa q)^2) and transforming back gives
// a' + i b' (a'' + i b'') directly -- no unpacking.  Eight threads share one packed line: thread t holds the samples
// n = t + 8 n2, does a radix-8 DFT in registers, exchanges through shared memory (__syncwarp only: the eight threads sit
// in one warp), does the second radix-8 pass and ends up with the modes k = t + 8 k1 -- the same stride-8 layout, so the
// inverse transforms are the same routine with conjugated twiddles.  Reading R12: modes q = -31 .. 31 and the Nyquist
// mode (first derivative 0, second derivative -(32 kappa)^2).
// ---------------------------------------------------------------------------------------------
struct cpx {
    double x, y;
};
__device__ __forceinline__ cpx operator+(cpx a, cpx b) { return { a.x + b.x, a.y + b.y }; }
__device__ __forceinline__ cpx operator-(cpx a, cpx b) { return { a.x - b.x, a.y - b.y }; }
__device__ __forceinline__ cpx cmul(cpx a, cpx b) { return { a.x * b.x - a.y * b.y, a.x * b.y + a.y * b.x }; }
// multiplication by exp(S i pi/2) = S i  (S = -1: forward transform, +1: inverse)
template <int S>
__device__ __forceinline__ cpx mul_si(cpx a)
{
    return S > 0 ? cpx{ -a.y, a.x } : cpx{ a.y, -a.x };
}
// 4-point DFT in place, natural order: X[k] = sum_n c_n exp(S 2 pi i n k / 4)
template <int S>
__device__ __forceinline__ void dft4(cpx &c0, cpx &c1, cpx &c2, cpx &c3)
{
    const cpx e0 = c0 + c2, e1 = c0 - c2, o0 = c1 + c3, o1 = mul_si<S>(c1 - c3);
    c0 = e0 + o0; c2 = e0 - o0; c1 = e1 + o1; c3 = e1 - o1;
}
// 8-point DFT in place, natural order: X[k] = sum_n x_n exp(S 2 pi i n k / 8)
template <int S>
__device__ __forceinline__ void dft8(cpx (&x)[8])
{
    constexpr double h = 0.70710678118654752440;      // sqrt(1/2)
    cpx a0 = x[0] + x[4], a1 = x[1] + x[5], a2 = x[2] + x[6], a3 = x[3] + x[7];
    const cpx d0 = x[0] - x[4], d1 = x[1] - x[5], d2 = x[2] - x[6], d3 = x[3] - x[7];
    // b_j = d_j W8^j, W8 = exp(S i pi/4) = h (1 + S i)
    cpx b0 = d0;
    cpx b1 = { h * (d1.x - S * d1.y), h * (d1.y + S * d1.x) };
    cpx b2 = mul_si<S>(d2);
    cpx b3 = { h * (-d3.x - S * d3.y), h * (-d3.y + S * d3.x) };
    dft4<S>(a0, a1, a2, a3);
    dft4<S>(b0, b1, b2, b3);
    x[0] = a0; x[2] = a1; x[4] = a2; x[6] = a3;
    x[1] = b0; x[3] = b1; x[5] = b2; x[7] = b3;
}
// 64-point transform of one packed line shared by 8 threads; in and out: thread t holds elements t + 8 m, m = 0..7.
// tw[m] = exp(-2 pi i t m / 64) (forward twiddles of this thread); ex = this line's exchange buffer (8 x 9 cpx).
template <int S>
__device__ __forceinline__ void fft64(cpx (&x)[8], const cpx (&tw)[8], cpx *ex, int t)
{
    dft8<S>(x);
#pragma unroll
    for (int k2 = 0; k2 < 8; ++k2) {
        const cpx w = S < 0 ? tw[k2] : cpx{ tw[k2].x, -tw[k2].y };
        ex[k2 * 9 + t] = k2 == 0 ? x[0] : cmul(x[k2], w);
    }
    __syncwarp();
#pragma unroll
    for (int n1 = 0; n1 < 8; ++n1) x[n1] = ex[t * 9 + n1];
    __syncwarp();
    dft8<S>(x);
}

constexpr int FFT_N = 64, FFT_PITCH = 33, FFT_LINES = 32;     // lines per CTA; staging rows padded against bank conflicts
// Grid: (R tile, Z row, job).  Measured alternatives, both slower: the job index fastest (so that the quantities of the
// same lines run together and share their reads in L2: +0.3 ms per step) and one CTA working through all quantities of
// its lines (+0.8 ms).
template <bool WANT2>
__global__ void __launch_bounds__(128) phi_fft64_kernel(const __grid_constant__ SpecArgs a, int job_base)
{
    __shared__ double sv[FFT_N * FFT_PITCH];                  // samples, then the first derivative
    // exchange buffers, one per packed line (8 x 9 cpx); once the transforms are done the same storage takes the
    // second derivative (FFT_N * FFT_PITCH doubles)
    __shared__ __align__(16) double sbuf[(FFT_LINES / 2) * 72 * 2];
    static_assert((FFT_LINES / 2) * 72 * 2 >= FFT_N * FFT_PITCH, "second-derivative staging fits the exchange storage");
    cpx *sex = reinterpret_cast<cpx *>(sbuf);
    double *s2 = sbuf;
    const Layout &L = a.L;
    const int tid = threadIdx.x, tx = tid & 31, ty = tid >> 5;
    const int i = 2 + blockIdx.x * 32 + tx, k = 2 + blockIdx.y;
    const bool valid = i <= L.nR - 3;
    const long long o2 = (long long)k * L.pR + (LP + min(i, L.nR - 3));
    const int job = job_base + blockIdx.z;
    const int pair = tid >> 3, t = tid & 7;                   // packed line (R nodes 2 pair, 2 pair + 1) and slot in it
    cpx tw[8];
#pragma unroll
    for (int m = 0; m < 8; ++m) {
        double sn, cs;
        sincospi(-(double)(t * m) / 32.0, &sn, &cs);
        tw[m] = { cs, sn };
    }
    const double kap = 6.283185307179586476925286766559 / a.ph.Lphi;
    int out1, out2;
    spec_stage(a, job, o2, sv, FFT_PITCH, tx, ty, 4, out1, out2);
    const bool want2 = WANT2 && out2 >= 0;
    __syncthreads();

    cpx z[8];
#pragma unroll
    for (int m = 0; m < 8; ++m) {
        z[m].x = sv[(t + 8 * m) * FFT_PITCH + 2 * pair];
        z[m].y = sv[(t + 8 * m) * FFT_PITCH + 2 * pair + 1];
    }
    cpx *ex = sex + pair * 72;
    fft64<-1>(z, tw, ex, t);
    // mode k = t + 8 m: signed wavenumber q (Nyquist: first derivative 0); 1/N of the inverse transform folded in
    cpx d1[8], d2[8];
#pragma unroll
    for (int m = 0; m < 8; ++m) {
        const int kk = t + 8 * m;
        const double q = kap * (double)(kk < 32 ? kk : kk - 64);
        const double w1 = kk == 32 ? 0.0 : q * (1.0 / 64.0), w2 = -(q * q) * (1.0 / 64.0);
        d1[m] = { -w1 * z[m].y, w1 * z[m].x };
        if (WANT2) d2[m] = { w2 * z[m].x, w2 * z[m].y };
    }
    fft64<1>(d1, tw, ex, t);
    if (WANT2) fft64<1>(d2, tw, ex, t);
    __syncthreads();                                          // every thread has taken its samples out of sv
#pragma unroll
    for (int m = 0; m < 8; ++m) {
        sv[(t + 8 * m) * FFT_PITCH + 2 * pair] = d1[m].x;
        sv[(t + 8 * m) * FFT_PITCH + 2 * pair + 1] = d1[m].y;
        if (WANT2) {
            s2[(t + 8 * m) * FFT_PITCH + 2 * pair] = d2[m].x;
            s2[(t + 8 * m) * FFT_PITCH + 2 * pair + 1] = d2[m].y;
        }
    }
    __syncthreads();
    if (valid) {
        for (int j = ty; j < FFT_N; j += 4) {
            const long long g = (long long)j * L.plane + o2;
            a.out[(long long)out1 * L.field + g] = sv[j * FFT_PITCH + tx];
            if (want2) a.out[(long long)out2 * L.field + g] = s2[j * FFT_PITCH + tx];
        }
    }
}

template <bool WANT2>
static cudaError_t launch_phi_jobs(const SpecArgs &a, int job_base, int jobs, cudaStream_t s, bool configure)
{
    auto kern = phi_spectral_kernel<WANT2>;
    if (configure)
        return cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                    (int)((SPEC_MAX_NPHI * 32 + 2 * SPEC_MAX_NPHI) * sizeof(double)));
    const int N = a.L.nphi;
    if (N == FFT_N) {
        dim3 grid((a.L.nR - 4 + 31) / 32, a.L.nZ - 4, jobs);
        phi_fft64_kernel<WANT2><<<grid, 128, 0, s>>>(a, job_base);
        return cudaGetLastError();
    }
    const int groups = (N + CLT_SPEC_NQ - 1) / CLT_SPEC_NQ;
    dim3 block(32, groups < 16 ? groups : 16, 1);
    dim3 grid((a.L.nR - 4 + 31) / 32, a.L.nZ - 4, jobs);
    const size_t smem = ((size_t)N * 32 + 2 * (size_t)N) * sizeof(double);
    kern<<<grid, block, smem, s>>>(a, job_base);
    return cudaGetLastError();
}

// mode 0: one launch (first derivatives of B1_R, B1_Z [, p1]); mode 1: two launches (the five fluid fields with
// both derivatives; E1_R, E1_Z with first derivatives only)
cudaError_t launch_phi_spectral(const SpecArgs &a, cudaStream_t s, bool configure)
{
    if (configure) {
        cudaError_t e = launch_phi_jobs<true>(a, 0, 0, s, true);
        return e != cudaSuccess ? e : launch_phi_jobs<false>(a, 0, 0, s, true);
    }
    if (a.mode == 0) return launch_phi_jobs<false>(a, 0, a.hall ? 3 : 2, s, false);
    cudaError_t e = launch_phi_jobs<true>(a, 0, 5, s, false);
    if (e != cudaSuccess) return e;
    return launch_phi_jobs<false>(a, 5, 2, s, false);
}

// ---------------------------------------------------------------------------------------------
// Axisymmetric tables (once per clt_set_equilibrium): J0 = curl_c B0 etc.
// ---------------------------------------------------------------------------------------------
__global__ void tables_kernel(Layout L, Phys ph, double *tab, const double *R, const double *invR)
{
    const int i = blockIdx.x * blockDim.x + threadIdx.x, k = blockIdx.y * blockDim.y + threadIdx.y;
    if (i >= L.nR || k >= L.nZ) return;
    const long long o = (long long)k * L.pR + (LP + i);
    auto T = [&](int t) -> double * { return tab + (long long)t * L.plane; };
    const double v0R = T(T_V0R)[o], v0P = T(T_V0P)[o], v0Z = T(T_V0Z)[o];
    const double B0R = T(T_B0R)[o], B0P = T(T_B0P)[o], B0Z = T(T_B0Z)[o];
    // E0 = v0 x B0 at every node (E1 is needed on the boundary layers too)
    T(T_E0R)[o] = v0P * B0Z - v0Z * B0P;
    T(T_E0P)[o] = v0Z * B0R - v0R * B0Z;
    T(T_E0Z)[o] = v0R * B0P - v0P * B0R;
    const bool interior = i >= 2 && i <= L.nR - 3 && k >= 2 && k <= L.nZ - 3;
    double out[T_COUNT];
    for (int t = T_J0R; t < T_COUNT; ++t) out[t] = 0.0;
    if (interior) {
        const int pR = L.pR;
        auto dR = [&](int t) { const double *f = T(t) + o; return fd1(f[-2], f[-1], f[1], f[2]) * ph.cR1; };
        auto dZ = [&](int t) { const double *f = T(t) + o; return fd1(f[-2 * pR], f[-pR], f[pR], f[2 * pR]) * ph.cZ1; };
        const double iR = invR[i];
        const double *bp = T(T_B0P) + o;
        const double dR_RB0P = fd1(R[i - 2] * bp[-2], R[i - 1] * bp[-1], R[i + 1] * bp[1], R[i + 2] * bp[2]) * ph.cR1;
        out[T_J0R] = -dZ(T_B0P);
        out[T_J0P] = dZ(T_B0R) - dR(T_B0Z);
        out[T_J0Z] = dR_RB0P * iR;
        out[T_GR_RHO0] = dR(T_RHO0); out[T_GZ_RHO0] = dZ(T_RHO0);
        out[T_GR_P0] = dR(T_P0);     out[T_GZ_P0] = dZ(T_P0);
        const double gRR = dR(T_V0R), gZR = dZ(T_V0R), gRP = dR(T_V0P), gZP = dZ(T_V0P), gRZ = dR(T_V0Z), gZZ = dZ(T_V0Z);
        out[T_GR_V0R] = gRR; out[T_GZ_V0R] = gZR; out[T_GR_V0P] = gRP; out[T_GZ_V0P] = gZP;
        out[T_GR_V0Z] = gRZ; out[T_GZ_V0Z] = gZZ;
        out[T_DIVV0] = gRR + v0R * iR + gZZ;
        out[T_A0R] = v0R * gRR + v0Z * gZR - v0P * v0P * iR;
        out[T_A0P] = v0R * gRP + v0Z * gZP + v0P * v0R * iR;
        out[T_A0Z] = v0R * gRZ + v0Z * gZZ;
    }
    for (int t = T_J0R; t < T_COUNT; ++t)
        if (t < T_E0R || t > T_E0Z) T(t)[o] = out[t];
}

cudaError_t launch_tables(const Layout &L, const Phys &ph, double *tab, const double *R, const double *invR,
                          cudaStream_t s)
{
    dim3 block(32, 8), grid((L.nR + 31) / 32, (L.nZ + 7) / 8);
    tables_kernel<<<grid, block, 0, s>>>(L, ph, tab, R, invR);
    return cudaGetLastError();
}

// Does the reference state move?  One block scans v0 (three tables) and raises *flag: selects the v0 = 0
// specialisation of the kernels without a synchronous copy of the tables to the host.
__global__ void __launch_bounds__(1024) any_nonzero_kernel(const double *x, long long n, int *flag)
{
    int mine = 0;
    for (long long q = threadIdx.x; q < n; q += blockDim.x) mine |= (x[q] != 0.0);
    const int any = __syncthreads_or(mine);
    if (threadIdx.x == 0) *flag = any;
}

cudaError_t launch_any_nonzero(const double *x, long long n, int *flag, cudaStream_t s)
{
    any_nonzero_kernel<<<1, 1024, 0, s>>>(x, n, flag);
    return cudaGetLastError();
}

// ---------------------------------------------------------------------------------------------
// a1: boundary layers.  The two outer node layers in R and Z hold the values given to
// clt_set_state in every RK buffer (L123, L187-189); the step kernels never write them.
// ---------------------------------------------------------------------------------------------
__device__ __forceinline__ bool boundary_node(const Layout &L, long long n, int &i, int &k, long long &row)
{
    // enumerate boundary nodes of one plane: 4 full rows (k = 0,1,nZ-2,nZ-1) then 4 columns of the other rows
    const long long per_plane = 4LL * L.nR + 4LL * (L.nZ - 4);
    row = n / per_plane;               // (field, phi plane) index
    const long long r = n % per_plane;
    if (r < 4LL * L.nR) {
        const int kk = (int)(r / L.nR);
        k = kk < 2 ? kk : L.nZ - 4 + kk;
        i = (int)(r % L.nR);
    } else {
        const long long t = r - 4LL * L.nR;
        k = 2 + (int)(t >> 2);
        const int c = (int)(t & 3);
        i = c < 2 ? c : L.nR - 4 + c;
    }
    return true;
}

__global__ void copy_boundary_kernel(Layout L, long long total, const double *src, double *d0, double *d1, double *d2)
{
    for (long long n = blockIdx.x * (long long)blockDim.x + threadIdx.x; n < total;
         n += (long long)gridDim.x * blockDim.x) {
        int i, k;
        long long row;
        boundary_node(L, n, i, k, row);
        const long long o = row * L.plane + (long long)k * L.pR + (LP + i);
        const double v = src ? src[o] : 0.0;
        if (d0) d0[o] = v;
        if (d1) d1[o] = v;
        if (d2) d2[o] = v;
    }
}

cudaError_t launch_copy_boundary(const Layout &L, int nfields, const double *src, double *d0, double *d1, double *d2,
                                 int sm_count, cudaStream_t s)
{
    const long long total = (long long)nfields * L.nphi * (4LL * L.nR + 4LL * (L.nZ - 4));
    const int block = 256;
    const long long want = (total + block - 1) / block, cap = (long long)(sm_count > 0 ? sm_count : 148) * 16;
    const int grid = (int)(want < cap ? want : cap);
    copy_boundary_kernel<<<grid, block, 0, s>>>(L, total, src, d0, d1, d2);
    return cudaGetLastError();
}

// NEXT-4: ghost rows of a neighbouring slab, straight from its buffer into this one (8 fields x nphi planes x nrows rows
// of nR nodes; the two layouts differ only in nZ)
__global__ void push_rows_kernel(Layout Ls, const double *src, int k0s, Layout Ld, double *dst, int k0d, int nrows, long long total)
{
    const int nR = Ls.nR;
    for (long long n = blockIdx.x * (long long)blockDim.x + threadIdx.x; n < total; n += (long long)gridDim.x * blockDim.x) {
        const int i = (int)(n % nR);
        const long long r = n / nR;
        const int row = (int)(r % nrows);
        const long long slice = r / nrows;                   // field * nphi + plane
        dst[slice * Ld.plane + (long long)(k0d + row) * Ld.pR + (LP + i)] =
            src[slice * Ls.plane + (long long)(k0s + row) * Ls.pR + (LP + i)];
    }
}

cudaError_t launch_push_rows(const Layout &Ls, const double *src, int k0s, const Layout &Ld, double *dst, int k0d, int nrows,
                             int sm_count, cudaStream_t s)
{
    const long long total = 8LL * Ls.nphi * nrows * Ls.nR;
    const int block = 256;
    const long long want = (total + block - 1) / block, cap = (long long)(sm_count > 0 ? sm_count : 148) * 8;
    push_rows_kernel<<<(int)(want < cap ? want : cap), block, 0, s>>>(Ls, src, k0s, Ld, dst, k0d, nrows, total);
    return cudaGetLastError();
}

cudaError_t launch_zero_boundary(const Layout &L, int nfields, double *dst, int sm_count, cudaStream_t s)
{
    return launch_copy_boundary(L, nfields, nullptr, dst, nullptr, nullptr, sm_count, s);
}

// ---------------------------------------------------------------------------------------------
// a7 diagnostics (L139, L149, L430) and the SETDT minimum (Fig. 4).
// A CTA owns 32 neighbouring R nodes of one Z row and all nphi planes: thread (tx, g) marches the g-th of DG_G
// contiguous phi chunks (so 8 x more threads stream than one per (R, Z) column, and B_phi's phi neighbours for
// div_c B come from a 5-deep register pipeline instead of being read five times).  The chunk partials -- the
// Fourier sums of the n = 1 harmonic have to be complete before they are squared -- meet in shared memory and
// are combined in a fixed order; warp shuffles reduce over R; the block partials are combined in a fixed order
// by a second, single-block kernel (deterministic).
// SETDT is regrouped (rounding order only): a node's three cell-crossing times become the rates (|v_d| + c)/h_d with
// h_R = |R_i - R_{i-1}| as in Fig. 4; the maximum is taken over the nodes and dt = min(100, cfl / max rate) once.
// ---------------------------------------------------------------------------------------------
constexpr int DG_BX = 32, DG_G = 8, DG_N = 6;   // kinetic, magnetic, magnetic_pert, magnetic_n1, max divB, max rate
constexpr int DG_Q = 11;                        // per-thread partials: ke, me, mep, fa[3], fb[3], mdiv, rate

__device__ __forceinline__ double warp_sum(double v)
{
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
    return v;
}
__device__ __forceinline__ double warp_max(double v)
{
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v = fmax(v, __shfl_xor_sync(0xffffffffu, v, o));
    return v;
}

__global__ void __launch_bounds__(DG_BX *DG_G, 2) diag_kernel(const __grid_constant__ DiagArgs a)
{
    const Layout &L = a.L;
    const Phys &ph = a.ph;
    const int tx = threadIdx.x, g = threadIdx.y, n = L.nphi;
    const int i = 2 + blockIdx.x * DG_BX + tx, k = 2 + blockIdx.y;
    const int ja = (int)(((long long)n * g) / DG_G), jb = (int)(((long long)n * (g + 1)) / DG_G);
    const bool valid = i <= L.nR - 3 && k >= a.k_first && k <= a.k_last;
    const bool deep = valid && i >= 4 && i <= L.nR - 5 && k >= a.kd_first && k <= a.kd_last;
    const double inf = __longlong_as_double(0x7ff0000000000000LL);
    double ke = 0.0, me = 0.0, mep = 0.0, mdiv = 0.0, rate = 0.0;
    double fa[3] = { 0, 0, 0 }, fb[3] = { 0, 0, 0 };
    if (valid && ja < jb) {
        const long long o = (long long)k * L.pR + (LP + i);
        const double Ri = a.R[i], iR = a.invR[i];
        const double b0R = a.tab[T_B0R * L.plane + o], b0P = a.tab[T_B0P * L.plane + o], b0Z = a.tab[T_B0Z * L.plane + o];
        const double ihR = 1.0 / fabs(Ri - a.R[i - 1]), ihP = 1.0 / fabs(Ri * ph.dphi);
        const double *Bp = a.U + 6 * L.field + o;
        const bool pipe = a.spec_c1 == nullptr;     // finite differences: B_phi of planes j-2 .. j+2 in registers
        double bp[5] = { 0, 0, 0, 0, 0 };
        if (pipe) {
#pragma unroll
            for (int d = 0; d < 4; ++d) bp[d + 1] = Bp[(long long)wrap_phi(ja - 2 + d, n) * L.plane];
        }
        // Everything one node-plane needs is requested in ONE batch (own values, B_phi of plane j+2, the R and Z stencil
        // neighbours of div_c B -- valid addresses for every interior node, used or not): the kernel is a latency chain
        // otherwise (ncu: 65 % of the warp time waiting for three dependent load batches per plane).
        struct Batch {
            double rho, p, vR, vP, vZ, BR, BZ, bpn, br[4], bz[4];
        };
        const double rr[4] = { a.R[i - 2], a.R[i - 1], a.R[i + 1], a.R[i + 2] };
        auto request = [&](int j) {
            Batch q;
            const long long gq = (long long)j * L.plane + o;
            q.rho = a.U[gq]; q.p = a.U[L.field + gq];
            q.vR = a.U[2 * L.field + gq]; q.vP = a.U[3 * L.field + gq]; q.vZ = a.U[4 * L.field + gq];
            q.BR = a.U[5 * L.field + gq]; q.BZ = a.U[7 * L.field + gq];
            q.bpn = Bp[(long long)(pipe ? wrap_phi(j + 2, n) : j) * L.plane];     // FD: plane j+2 of the pipeline; spectral: B_phi itself
            const double *br = a.U + 5 * L.field + gq, *bz = a.U + 7 * L.field + gq;
            q.br[0] = br[-2]; q.br[1] = br[-1]; q.br[2] = br[1]; q.br[3] = br[2];
            q.bz[0] = bz[-2 * L.pR]; q.bz[1] = bz[-L.pR]; q.bz[2] = bz[L.pR]; q.bz[3] = bz[2 * L.pR];
            return q;
        };
#pragma unroll 1
        for (int j = ja; j < jb; ++j) {
            const Batch q = request(j);
            const double rho = q.rho, p = q.p, vR = q.vR, vP = q.vP, vZ = q.vZ, BR = q.BR, BZ = q.BZ;
            double BP;
            if (pipe) {
#pragma unroll
                for (int d = 0; d < 4; ++d) bp[d] = bp[d + 1];
                bp[4] = q.bpn;
                BP = bp[2];
            } else {
                BP = q.bpn;
            }
            const double b2 = BR * BR + BP * BP + BZ * BZ;
            ke += 0.5 * rho * (vR * vR + vP * vP + vZ * vZ);
            me += 0.5 * b2;
            const double b1[3] = { BR - b0R, BP - b0P, BZ - b0Z };
            mep += 0.5 * (b1[0] * b1[0] + b1[1] * b1[1] + b1[2] * b1[2]);
            const double c = a.cs[j], s = a.cs[n + j];
#pragma unroll
            for (int d = 0; d < 3; ++d) { fa[d] += b1[d] * c; fb[d] += b1[d] * s; }
            // SETDT, Fig. 4: signal speed and the three rates
            const double cf = sqrt(fabs((ph.gamma * p + b2) / rho));
            const double rR = (fabs(vR) + cf) * ihR, rZ = (fabs(vZ) + cf) * a.ihZ, rP = (fabs(vP) + cf) * ihP;
            rate = fmax(rate, fmax(rP, fmax(rR, rZ)));
            if (!(rR + rP + rZ <= 1.79769313486231570815e308)) rate = inf;     // fmax drops NaN: mark a non-finite state
            if (deep) {
                // div_c B = d_R(R B_R)/R + d_phi B_phi / R + d_Z B_Z
                const double dRR = fd1(rr[0] * q.br[0], rr[1] * q.br[1], rr[2] * q.br[2], rr[3] * q.br[3]);
                double dPs;      // d_phi B_phi
                if (pipe) {
                    dPs = fd1(bp[0], bp[1], bp[3], bp[4]) * ph.cP1;
                } else {
                    dPs = 0.0;   // pseudo-spectral: paired circulant sum (B0_phi drops out of the differences)
                    for (int m = 1; m <= (n - 1) / 2; ++m)
                        dPs = fma(a.spec_c1[m], Bp[(long long)wrap_phi(j + m, n) * L.plane] - Bp[(long long)wrap_phi(j - m, n) * L.plane], dPs);
                }
                const double dZ = fd1(q.bz[0], q.bz[1], q.bz[2], q.bz[3]);
                mdiv = fmax(mdiv, fabs(dRR * ph.cR1 * iR + dPs * iR + dZ * ph.cZ1));
            }
        }
    }
    // phi chunks meet in shared memory; chunk 0's warp combines them in a fixed order
    __shared__ double sh[DG_G][DG_Q][DG_BX];
    {
        double (*m)[DG_BX] = sh[g];
        m[0][tx] = ke; m[1][tx] = me; m[2][tx] = mep;
#pragma unroll
        for (int d = 0; d < 3; ++d) { m[3 + d][tx] = fa[d]; m[6 + d][tx] = fb[d]; }
        m[9][tx] = mdiv; m[10][tx] = rate;
    }
    __syncthreads();
    if (g != 0) return;
    auto sum_chunks = [&](int q) {
        double v = sh[0][q][tx];
#pragma unroll
        for (int w = 1; w < DG_G; ++w) v += sh[w][q][tx];
        return v;
    };
    auto max_chunks = [&](int q) {
        double v = sh[0][q][tx];
#pragma unroll
        for (int w = 1; w < DG_G; ++w) v = fmax(v, sh[w][q][tx]);
        return v;
    };
    double out[DG_N] = { 0, 0, 0, 0, 0, 0 };
    if (valid) {
        const double Ri = a.R[i];
        const double w = Ri * ph.dR * ph.dphi * ph.dZ;
        out[0] = sum_chunks(0) * w; out[1] = sum_chunks(1) * w; out[2] = sum_chunks(2) * w;
        const double sc = 2.0 / (double)n;
        double e1 = 0.0;
#pragma unroll
        for (int d = 0; d < 3; ++d) { const double A = sum_chunks(3 + d) * sc, B = sum_chunks(6 + d) * sc; e1 += A * A + B * B; }
        out[3] = 0.25 * e1 * (Ri * ph.dR * ph.dZ * ph.Lphi);
        out[4] = max_chunks(9); out[5] = max_chunks(10);
    }
#pragma unroll
    for (int q = 0; q < 4; ++q) out[q] = warp_sum(out[q]);
    out[4] = warp_max(out[4]); out[5] = warp_max(out[5]);
    if (tx == 0) {
        double *dst = a.partial + (long long)(blockIdx.y * gridDim.x + blockIdx.x) * DG_N;
#pragma unroll
        for (int q = 0; q < DG_N; ++q) dst[q] = out[q];
    }
}

// TMA-fed variant of the reduction (finite-difference phi scheme; the default): the curl kernel's sweep.  A CTA owns a
// 32 x DGT_TZ tile and marches over all planes; one bulk copy per plane brings the 8 fields of the tile with its halo into a
// DGT_NS-slot ring three planes ahead, so nothing waits for HBM in front of the square root and the division of SETDT;
// B_phi's phi neighbours sit in a register pipeline, the R / Z neighbours of div_c B come from the tile, and a thread sees
// all planes of its node: the Fourier sums of the n = 1 harmonic are complete in its registers.
constexpr int DGT_TZ = 8, DGT_NS = 4;
struct DiagTmaSmem {
    static constexpr int HT = (DGT_TZ + 4) * SW;
    alignas(128) double raw[DGT_NS][8][HT];
    alignas(8) unsigned long long full[DGT_NS];
    double red[DGT_TZ][DG_N];
};

__global__ void __launch_bounds__(TR *DGT_TZ, 2) diag_tma_kernel(const __grid_constant__ DiagArgs a, const __grid_constant__ CUtensorMap tmU)
{
    extern __shared__ __align__(128) unsigned char smem_raw[];
    DiagTmaSmem &S = *reinterpret_cast<DiagTmaSmem *>(smem_raw);
    constexpr int HT = DiagTmaSmem::HT, NS = DGT_NS, TZ = DGT_TZ;
    static_assert(HT % 16 == 0, "a box that spans the field axis fills a ring slot densely");
    const Layout &L = a.L;
    const Phys &ph = a.ph;
    const int tx = threadIdx.x, ty = threadIdx.y, tid = ty * TR + tx, n = L.nphi;
    const int i0 = 2 + TR * blockIdx.x, k0 = 2 + TZ * blockIdx.y;
    const int i = i0 + tx, k = k0 + ty;
    const bool valid = i <= L.nR - 3 && k <= L.nZ - 3 && k >= a.k_first && k <= a.k_last;
    const bool deep = valid && i >= 4 && i <= L.nR - 5 && k >= a.kd_first && k <= a.kd_last;
    const int ic = min(i, L.nR - 3), kc = min(k, L.nZ - 3);
    const long long o = (long long)kc * L.pR + (LP + ic);
    const int cs = (ty + 2) * SW + (tx + 2);
    const int total = n + 4;                                  // planes -2 .. n+1

    if (tid == 0) {
        for (int q = 0; q < NS; ++q) mbar_init(&S.full[q], 1);
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
        asm volatile("prefetch.tensormap [%0];" ::"l"(&tmU) : "memory");
    }
    __syncthreads();
    auto issue = [&](int q) {                                 // plane number q counts from plane -2
        const int st = q % NS;
        mbar_expect_tx(&S.full[st], (unsigned)(8 * HT * sizeof(double)));
        tma_load_4d(&S.raw[st][0][0], &tmU, LP + i0 - 2, k0 - 2, wrap_phi(q - 2, n), 0, &S.full[st]);
    };
    if (tid == 0)
        for (int q = 0; q < NS && q < total; ++q) issue(q);

    const double inf = __longlong_as_double(0x7ff0000000000000LL);
    const double Ri = a.R[ic], iR = a.invR[ic];
    const double b0R = a.tab[T_B0R * L.plane + o], b0P = a.tab[T_B0P * L.plane + o], b0Z = a.tab[T_B0Z * L.plane + o];
    const double ihR = 1.0 / fabs(Ri - a.R[ic - 1]), ihP = 1.0 / fabs(Ri * ph.dphi);
    const double rr[4] = { a.R[ic - 2], a.R[ic - 1], a.R[ic + 1], a.R[ic + 2] };
    double ke = 0.0, me = 0.0, mep = 0.0, mdiv = 0.0, rate = 0.0;
    double fa[3] = { 0, 0, 0 }, fb[3] = { 0, 0, 0 };
    double bp[5] = { 0, 0, 0, 0, 0 };                         // B_phi of planes j-2 .. j+2 at the own node
#pragma unroll 1
    for (int q = 0; q < 4; ++q) {
        mbar_wait(&S.full[q % NS], (unsigned)((q / NS) & 1));
        bp[q + 1] = S.raw[q % NS][6][cs];
    }
    __syncthreads();                                          // planes 0 and 1 are never centre planes: recycle their slots
    if (tid == 0) {
        if (NS < total) issue(NS);
        if (NS + 1 < total) issue(NS + 1);
    }
#pragma unroll 1
    for (int j = 0; j < n; ++j) {
        const int nc = j + 2;                                 // plane number of the centre plane
        mbar_wait(&S.full[(nc + 2) % NS], (unsigned)(((nc + 2) / NS) & 1));
#pragma unroll
        for (int d = 0; d < 4; ++d) bp[d] = bp[d + 1];
        bp[4] = S.raw[(nc + 2) % NS][6][cs];
        const double (*f)[HT] = S.raw[nc % NS];
        const double rho = f[0][cs], p = f[1][cs], vR = f[2][cs], vP = f[3][cs], vZ = f[4][cs], BR = f[5][cs], BZ = f[7][cs];
        const double BP = bp[2];
        if (valid) {
            const double b2 = BR * BR + BP * BP + BZ * BZ;
            ke += 0.5 * rho * (vR * vR + vP * vP + vZ * vZ);
            me += 0.5 * b2;
            const double b1[3] = { BR - b0R, BP - b0P, BZ - b0Z };
            mep += 0.5 * (b1[0] * b1[0] + b1[1] * b1[1] + b1[2] * b1[2]);
            const double c = a.cs[j], s = a.cs[n + j];
#pragma unroll
            for (int d = 0; d < 3; ++d) { fa[d] += b1[d] * c; fb[d] += b1[d] * s; }
            // SETDT, Fig. 4: signal speed and the three rates
            const double cf = sqrt(fabs((ph.gamma * p + b2) / rho));
            const double rR = (fabs(vR) + cf) * ihR, rZ = (fabs(vZ) + cf) * a.ihZ, rP = (fabs(vP) + cf) * ihP;
            rate = fmax(rate, fmax(rP, fmax(rR, rZ)));
            if (!(rR + rP + rZ <= 1.79769313486231570815e308)) rate = inf;     // fmax drops NaN: mark a non-finite state
            if (deep) {
                // div_c B = d_R(R B_R)/R + d_phi B_phi / R + d_Z B_Z
                const double *br = &f[5][cs], *bz = &f[7][cs];
                const double dRR = fd1(rr[0] * br[-2], rr[1] * br[-1], rr[2] * br[1], rr[3] * br[2]);
                const double dPs = fd1(bp[0], bp[1], bp[3], bp[4]) * ph.cP1;
                const double dZ = fd1(bz[-2 * SW], bz[-SW], bz[SW], bz[2 * SW]);
                mdiv = fmax(mdiv, fabs(dRR * ph.cR1 * iR + dPs * iR + dZ * ph.cZ1));
            }
        }
        __syncthreads();                                      // the centre plane's slot is free again
        if (tid == 0 && nc + NS < total) issue(nc + NS);
    }
    double out[DG_N] = { 0, 0, 0, 0, 0, 0 };
    if (valid) {
        const double w = Ri * ph.dR * ph.dphi * ph.dZ;
        out[0] = ke * w; out[1] = me * w; out[2] = mep * w;
        const double sc = 2.0 / (double)n;
        double e1 = 0.0;
#pragma unroll
        for (int d = 0; d < 3; ++d) { const double A = fa[d] * sc, B = fb[d] * sc; e1 += A * A + B * B; }
        out[3] = 0.25 * e1 * (Ri * ph.dR * ph.dZ * ph.Lphi);
        out[4] = mdiv; out[5] = rate;
    }
#pragma unroll
    for (int q = 0; q < 4; ++q) out[q] = warp_sum(out[q]);
    out[4] = warp_max(out[4]); out[5] = warp_max(out[5]);
    if (tx == 0)
        for (int q = 0; q < DG_N; ++q) S.red[ty][q] = out[q];
    __syncthreads();
    if (tid == 0) {                                           // warps in a fixed order (deterministic)
        double r[DG_N] = { 0, 0, 0, 0, 0, 0 };
        for (int w = 0; w < TZ; ++w) {
            for (int q = 0; q < 4; ++q) r[q] += S.red[w][q];
            r[4] = fmax(r[4], S.red[w][4]); r[5] = fmax(r[5], S.red[w][5]);
        }
        double *dst = a.partial + (long long)(blockIdx.y * gridDim.x + blockIdx.x) * DG_N;
        for (int q = 0; q < DG_N; ++q) dst[q] = r[q];
    }
}

// result = { kinetic, magnetic, magnetic_pert, magnetic_n1, max |div_c B|, dt = min(100, cfl / max rate) }; an infinite
// rate (non-finite state) gives dt = 0
__global__ void __launch_bounds__(256) diag_final_kernel(const double *partial, int nblocks, double cfl, double *result)
{
    __shared__ double red[8][DG_N];
    double acc[DG_N] = { 0, 0, 0, 0, 0, 0 };
    for (int b = threadIdx.x; b < nblocks; b += 256) {
        const double *p = partial + (long long)b * DG_N;
        for (int q = 0; q < 4; ++q) acc[q] += p[q];
        acc[4] = fmax(acc[4], p[4]);
        acc[5] = fmax(acc[5], p[5]);
    }
    for (int q = 0; q < 4; ++q) acc[q] = warp_sum(acc[q]);
    acc[4] = warp_max(acc[4]);
    acc[5] = warp_max(acc[5]);
    const int w = threadIdx.x >> 5;
    if ((threadIdx.x & 31) == 0)
        for (int q = 0; q < DG_N; ++q) red[w][q] = acc[q];
    __syncthreads();
    if (threadIdx.x == 0) {
        double out[DG_N] = { 0, 0, 0, 0, 0, 0 };
        for (int ww = 0; ww < 8; ++ww) {
            for (int q = 0; q < 4; ++q) out[q] += red[ww][q];
            out[4] = fmax(out[4], red[ww][4]);
            out[5] = fmax(out[5], red[ww][5]);
        }
        out[5] = out[5] > 0.0 ? fmin(100.0, cfl / out[5]) : 100.0;      // Fig. 4: DT1 starts at 100
        for (int q = 0; q < DG_N; ++q) result[q] = out[q];
    }
}

int diag_blocks(const Layout &L)
{
    return ((L.nR - 4 + DG_BX - 1) / DG_BX) * (L.nZ - 4);
}

int diag_tma_tile_z() { return DGT_TZ; }

// tmU != nullptr (and the finite-difference phi scheme): the TMA-fed kernel; tmU maps the 8 fields of the state with box
// (TR+4, diag_tma_tile_z()+4, 1, 8).  configure = true: only the shared-memory opt-in.
cudaError_t launch_diag(const DiagArgs &a, int nblocks, double *result6, cudaStream_t s, const void *tmU, bool configure)
{
    if (configure)
        return cudaFuncSetAttribute(diag_tma_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sizeof(DiagTmaSmem));
    cudaError_t e;
    if (tmU && !a.spec_c1) {
        dim3 block(TR, DGT_TZ), grid((a.L.nR - 4 + TR - 1) / TR, (a.L.nZ - 4 + DGT_TZ - 1) / DGT_TZ);
        nblocks = (int)(grid.x * grid.y);
        diag_tma_kernel<<<grid, block, sizeof(DiagTmaSmem), s>>>(a, *reinterpret_cast<const CUtensorMap *>(tmU));
        e = cudaGetLastError();
    } else {
        dim3 block(DG_BX, DG_G), grid((a.L.nR - 4 + DG_BX - 1) / DG_BX, a.L.nZ - 4);
        diag_kernel<<<grid, block, 0, s>>>(a);
        e = cudaGetLastError();
    }
    if (e != cudaSuccess) return e;
    diag_final_kernel<<<1, 256, 0, s>>>(a.partial, nblocks, a.cfl, result6);
    return cudaGetLastError();
}

// ---------------------------------------------------------------------------------------------
// clt_diagnostics_static: the block partials of the diagnostics reduction in a file-scope device array instead of the
// caller's workspace -- an entry point that needs no scratch from anybody (callers that cannot allocate: code under
// CUDA graph capture, tight serving loops).  DIAG_STATIC_MAX_BLOCKS x 6 doubles = 768 KiB, held by every GPU that loads
// the library until the process exits.  Nothing in it has to start at zero: every CTA of the reduction kernel writes
// its own 6 partials and the final kernel reads exactly the CTAs of its launch, so the contents a previous call left
// behind (even of a larger grid) are never read.  All calls on a device share the array: calls that overlap on the GPU
// (two streams) race.
// In host code the array's name is a host-side stand-in, not a device address: the address a kernel can use comes from
// cudaGetSymbolAddress, resolved per context at clt_create with the context's device current.
// ---------------------------------------------------------------------------------------------
constexpr int DIAG_STATIC_MAX_BLOCKS = 16384;
static __device__ __align__(256) double g_diag_static_partial[DIAG_STATIC_MAX_BLOCKS * DG_N];

cudaError_t diag_static_scratch(double **ptr, int *max_blocks)
{
    void *p = nullptr;
    cudaError_t e = cudaGetSymbolAddress(&p, g_diag_static_partial);      // the CURRENT device's copy of the array
    if (e != cudaSuccess) return e;
    *ptr = static_cast<double *>(p);
    *max_blocks = DIAG_STATIC_MAX_BLOCKS;
    return cudaSuccess;
}

// Opts every kernel with more than 48 KB of dynamic shared memory in on the CURRENT device (the attribute is per
// function and device).  Called by clt_create under the context's device, so nothing about it is process-global state.
cudaError_t configure_kernels()
{
    const RhsArgs ra{};
    const CurlArgs ca{};
    const SpecArgs sa{};
    const CUtensorMap tm{};
    for (int mode = RHS_MODE_K; mode <= RHS_MODE_S4; ++mode)
        for (int v0 = 0; v0 < 2; ++v0) {
            cudaError_t e = launch_rhs(ra, mode, v0 != 0, nullptr, true);
            if (e != cudaSuccess) return e;
            for (int hs = 0; hs < 8; ++hs) {
                e = launch_rhs_tma(ra, &tm, &tm, &tm, mode, v0 != 0, (hs & 1) != 0, (hs & 2) != 0, (hs & 4) != 0, nullptr, true);
                if (e != cudaSuccess) return e;
            }
        }
    for (int hs = 0; hs < 4; ++hs) {
        cudaError_t e = launch_curl_tma(ca, &tm, (hs & 1) != 0, (hs & 2) != 0, nullptr, true);
        if (e != cudaSuccess) return e;
    }
    cudaError_t e = launch_phi_spectral(sa, nullptr, true);
    if (e != cudaSuccess) return e;
    return launch_diag(DiagArgs{}, 0, nullptr, nullptr, nullptr, true);
}

}  // namespace clt
