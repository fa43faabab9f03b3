// m2l_math.cuh -- per-pair arithmetic of the multipole->local interaction, sm_100a.
//
// What it computes is defined in include/octo_fmm.h / DESIGN.md (section 2.2).
// How it computes it differs from the definition on purpose (this is the GPU formulation; the
// CPU oracle uses full tensors):
//   * The Green's-function derivative tensors D^(n) of -1/r are symmetric and TRACE-FREE, so only
//     2n+1 components of each are independent, and each is a radial factor d_n(r) times products
//     of R_i plus delta terms.  Source moments are reduced once per cell at staging time (trace
//     removed, multiplicity and (-1)^m/m! folded in).
//   * Correction on (m2l_pair_folded): no component of D2..D4 is formed; what a
//     source contributes is written as radial factors (with the source's mass folded in) times the
//     R-contractions S = q_jk R_j R_k, V_i = q_ij R_j, a = m1.R, and the correction goes through the
//     cubic form C = n_ijk R_i R_j R_k (c_i = d4 C R_i + 3 d3 Q_i).  86 DFMA + 38 DMUL + 14 DADD per pair.
//   * Correction off (m2l_pair component form): the components of D1..D3 with at most one z index
//     contracted with the reduced moments, grouped so that consecutive FMAs share an operand.
//   * Accumulators are the independent components of L (1 + 3 + 5 + 7) and the correction (3);
//     the dependent components (L2_zz, L3_xzz, L3_yzz, L3_zzz) are rebuilt once per cell.
//   * 1/r comes from MUFU.RSQ64H (rsqrt.approx.ftz.f64, ~2^-21) and ONE cubically convergent
//     correction step, y (1 + e/2 + 3e^2/8), e = 1 - r^2 y^2: relative error ~ (5/16) e^3 < 1e-18.
#pragma once

namespace octo {

// staged (internal) per-cell source components
enum {
    C_M0 = 0,
    C_M1X = 1, C_M1Y, C_M1Z,                               // -M1 (sign folded)
    C_QXX = 4, C_QXY, C_QXZ, C_QYY, C_QYZ,                 // reduced 1/2 M2
    C_OXXX = 9, C_OXXY, C_OXXZ, C_OXYY, C_OXYZ, C_OYYY, C_OYYZ,  // reduced -1/6 M3
    C_DX = 16, C_DY, C_DZ,                                 // centre-of-mass offset delta
    NCOMP = 19
};

// Accumulators of one target cell: the independent components of the trace-free L2 / L3, two partial sums of L0.
struct Acc {
    double l0, l0b; // two partial sums of L0
    double l1[3];
    double l2[5];   // xx xy xz yy yz
    double l3[7];   // xxx xxy xxz xyy xyz yyy yyz
    double c[3];    // correction to L1
};
constexpr int ACC_DOUBLES = 20;
static_assert(sizeof(Acc) == ACC_DOUBLES * sizeof(double), "Acc is a plain array of doubles");

__device__ __forceinline__ void acc_zero(Acc& a)
{
    a.l0 = 0.0;
    a.l0b = 0.0;
#pragma unroll
    for (int i = 0; i < 3; ++i) { a.l1[i] = 0.0; a.c[i] = 0.0; }
#pragma unroll
    for (int i = 0; i < 5; ++i) a.l2[i] = 0.0;
#pragma unroll
    for (int i = 0; i < 7; ++i) a.l3[i] = 0.0;
}

// constants that are not 32-bit immediates: as literals they are rebuilt by two moves per pair, from the constant bank
// they are an operand of the instruction
__constant__ double c_fold[2] = {-7.0 / 3.0, 0.375};

// 1/sqrt(x) to ~1 ulp for normal positive x
__device__ __forceinline__ double rsqrt_fast(double x)
{
    double y;
    asm("rsqrt.approx.ftz.f64 %0, %1;" : "=d"(y) : "d"(x));
    const double t = x * y;
    const double e = fma(-t, y, 1.0);
    const double p = fma(c_fold[1], e, 0.5);
    const double q = e * p;
    return fma(y, q, y);
}

// Reduce the 20 raw moments of a cell to the 16 staged source components (once per cell).
// With the correction ON the five quadrupole slots hold q~ = 1/2 x (trace-free part of M2) (for the evaluation
// through R-contractions in m2l_pair<true>) instead of the reduced 1/2 M2.
// The seven octupole slots hold, with the correction OFF, the reduced -1/6 M3 that contracts with the 7
// independent components of D3; with the correction ON, N' = -1/6 x (trace-free part of M3), components
// xxx xxy xxz xyy xyz yyy yyz -- the form the cubic-form evaluation of m2l_pair<true> needs.
__device__ __forceinline__ void reduce_moments(const double M[20], double* s, const bool corr)
{
    s[C_M0] = M[0];
    s[C_M1X] = -M[1];
    s[C_M1Y] = -M[2];
    s[C_M1Z] = -M[3];
    // M2: [xx xy xz yy yz zz] = M[4..9];  1/2 M2:D2 with D2_zz = -D2_xx - D2_yy
    s[C_QXX] = 0.5 * (M[4] - M[9]);
    s[C_QXY] = M[5];
    s[C_QXZ] = M[6];
    s[C_QYY] = 0.5 * (M[7] - M[9]);
    s[C_QYZ] = M[8];
    // M3: [xxx xxy xxz xyy xyz xzz yyy yyz yzz zzz] = M[10..19];  -1/6 M3:.D3 with
    // D3_xzz = -D3_xxx - D3_xyy, D3_yzz = -D3_xxy - D3_yyy, D3_zzz = -D3_xxz - D3_yyz
    s[C_OXXX] = -(M[10] - 3.0 * M[15]) * (1.0 / 6.0);
    s[C_OXXY] = -0.5 * (M[11] - M[18]);
    s[C_OXXZ] = -(3.0 * M[12] - M[19]) * (1.0 / 6.0);
    s[C_OXYY] = -0.5 * (M[13] - M[15]);
    s[C_OXYZ] = -M[14];
    s[C_OYYY] = -(M[16] - 3.0 * M[18]) * (1.0 / 6.0);
    s[C_OYYZ] = -(3.0 * M[17] - M[19]) * (1.0 / 6.0);
    if (corr) {
        // quadrupole slots: q~ = 1/2 x (trace-free part of M2), components xx xy xz yy yz
        const double tr3 = ((M[4] + M[7]) + M[9]) * (1.0 / 3.0);
        s[C_QXX] = 0.5 * (M[4] - tr3);
        s[C_QXY] = 0.5 * M[5];
        s[C_QXZ] = 0.5 * M[6];
        s[C_QYY] = 0.5 * (M[7] - tr3);
        s[C_QYZ] = 0.5 * M[8];
        // trace-free part: N_ijk = M_ijk - (d_ij t_k + d_ik t_j + d_jk t_i) / 5,  t_k = M_jjk
        const double tx = (M[10] + M[13]) + M[15], ty = (M[11] + M[16]) + M[18], tz = (M[12] + M[17]) + M[19];
        const double k = -1.0 / 6.0;
        s[C_OXXX] = k * (M[10] - 0.6 * tx);
        s[C_OXXY] = k * (M[11] - 0.2 * ty);
        s[C_OXXZ] = k * (M[12] - 0.2 * tz);
        s[C_OXYY] = k * (M[13] - 0.2 * tx);
        s[C_OXYZ] = k * M[14];
        s[C_OYYY] = k * (M[16] - 0.6 * ty);
        s[C_OYYZ] = k * (M[17] - 0.2 * tz);
    }
}

// Head of one ordered pair: 1/|R|.  Kept apart from the body so that the kernels can run the
// head of pair s+1 (a long dependent chain: r^2 -> MUFU -> correction step) under the body of pair s.
__device__ __forceinline__ double pair_head(const double x, const double y, const double z)
{
    const double r2 = fma(z, z, fma(y, y, x * x));
    return rsqrt_fast(r2);
}

// Body of one ordered pair with the correction ON.  Instead of generating the components of D2, D3, D4 and
// multiplying each by every source component, everything a source contributes is written as a radial factor times
// products of components of R, with the source's mass folded into the radial factors (e_n = M d_n):
//   L0   += -M w + d1 (m1.R) + d2 S + d3 C                 V_i = q~_ij R_j,  S = R.V,  Q_i = n_ijk R_j R_k,  C = R.Q
//   L1_i += k1 R_i + d1 m1_i + 2 d2 V_i                    k1 = c1 + d3 S
//   L2_ij += c1 d_ij + v_i R_j + h_j R_i                   c1 = e1 + d2 (m1.R),  c2 = e2 + d3 (m1.R),  h = d2 m1,  v = c2 R + h
//   L3_ijk += e2 (d_ij R_k + d_ik R_j + d_jk R_i) + e3 R_i R_j R_k
//   dL1_i += d4 C R_i + 3 d3 Q_i,  L0 += d3 C              n = N'_B - M_B (N'_A / M_A)   (L127)
// with m1 = -M1 (staged), q~ = 1/2 trace-free M2, N' = -1/6 trace-free M3, d1 = 1/r^3, d2 = -3/r^5, d3 = 15/r^7,
// d4 = -105/r^9.  These are the sums of the header of this file with D2_ij = d1 d_ij + d2 R_i R_j etc. multiplied out
// (the quadrupole and dipole parts use that D2 and D3 are trace-free).  What keeps the instruction count down:
//   - L3 is trace-free pair by pair (5 d2 + d3 r^2 = 0), so seven components carry it; the seven WITHOUT a repeated
//     triple index (xxy xxz xyy yyz xzz yzz xyz) need only f_ii = e3 R_i^2 + e2, never the 3 e2 of xxx, yyy, zzz;
//     acc_finish rebuilds xxx = -(xyy + xzz) etc.;
//   - the diagonal of L2 is completed per pair (c1 and c2 x^2 cancel to a large extent; summing them separately over
//     the list would lose those digits);
//   - a.c holds ONE THIRD of the correction, d3 Q_i + (d4 / 3) C R_i (acc_finish multiplies by 3); -7/3 and the 0.375
//     of rsqrt_fast come from the constant bank (c_fold), so no instruction rebuilds them.
// 130 FP64 instructions per pair with the dipole terms (82 DFMA, 35 DMUL, 13 DADD: 212 flop) and 113 without, against
// 157 / 129 for the component-by-component contraction; the oracle keeps the component form.
//
// ORDER OF THE STATEMENTS.  An FP64 instruction occupies the pipe for 2 cycles, and for 3 if all three of its source
// registers have to be read fresh (profiles/r02_sass_cost_model.md); an operand is free when the previous instruction
// of the warp read the same register in the same slot.  ptxas decides the final order, but it starts from the order of
// the source, so the statements below stand in the order that a search over dependency-respecting permutations found
// to give the fewest pipe cycles in the SASS of m2l_staged_kernel (python -m paper_2101_08226_b200.sass_cost_model:
// 41 of 82 DFMAs with three fresh registers instead of 59 for the "natural" order of the formulas above).  Each
// statement is one term of those formulas; names as above, n_ijk / p_ij (= x^2 - z^2, y^2 - z^2, 2xy, 2xz, 2yz) for
// the cubic form.
template <bool DIPOLE>
__device__ __forceinline__ void m2l_pair_folded(Acc& a, const double x, const double y, const double z, const double w,
                                                  const double (&s)[16], const double (&tA)[7])
{
    const double w2 = w * w;
    const double x2 = x + x;
    const double k3 = -3.0 * w2;
    const double m1y = DIPOLE ? s[C_M1Y] : 0.0;
    const double m0 = s[C_M0];
    const double qyz = s[C_QYZ];
    const double d1 = w * w2;
    const double y2 = y + y;
    const double d2 = d1 * k3;
    const double pyz = y2 * z;
    const double e2 = m0 * d2;
    const double qxy = s[C_QXY];
    const double pxz = x2 * z;
    const double nxxz = fma(-m0, tA[2], s[C_OXXZ]);
    const double k7 = c_fold[0] * w2;
    const double qxx = s[C_QXX];
    const double k5 = -5.0 * w2;
    const double d3 = d2 * k5;
    const double zz = z * z;
    if (DIPOLE) a.l1[1] = fma(d1, m1y, a.l1[1]);
    const double e3 = m0 * d3;
    const double m1x = DIPOLE ? s[C_M1X] : 0.0;
    const double hy = DIPOLE ? d2 * m1y : 0.0;
    const double e3y = e3 * y;
    const double qxz = s[C_QXZ];
    const double e3x = e3 * x;
    const double nxxy = fma(-m0, tA[1], s[C_OXXY]);
    const double qyy = s[C_QYY];
    const double fxx = fma(e3x, x, e2);
    const double nxyz = fma(-m0, tA[4], s[C_OXYZ]);
    const double fyy = fma(e3y, y, e2);
    const double nxyy = fma(-m0, tA[3], s[C_OXYY]);
    const double m1z = DIPOLE ? s[C_M1Z] : 0.0;
    const double qzz = -(qxx + qyy);
    const double e3z = e3 * z;
    const double e1 = m0 * d1;
    const double fzz = fma(e3z, z, e2);
    if (DIPOLE) a.l1[2] = fma(d1, m1z, a.l1[2]);
    const double ar = DIPOLE ? fma(m1z, z, fma(m1y, y, m1x * x)) : 0.0;
    const double d3k7 = d3 * k7;
    const double nxxx = fma(-m0, tA[0], s[C_OXXX]);
    const double pxy = x2 * y;
    const double pa = fma(x, x, -zz);
    const double c2 = DIPOLE ? fma(d3, ar, e2) : e2;
    const double nxzz = -(nxxx + nxyy);
    const double hx = DIPOLE ? d2 * m1x : 0.0;
    const double Vz = fma(qzz, z, fma(qyz, y, qxz * x));
    a.l3[2] = fma(fyy, x, a.l3[2]);
    const double nyyz = fma(-m0, tA[6], s[C_OYYZ]);
    a.l3[5] = fma(fzz, y, a.l3[5]);
    const double vx = DIPOLE ? fma(c2, x, hx) : c2 * x;
    const double vy = DIPOLE ? fma(c2, y, hy) : c2 * y;
    a.l2[1] = fma(vx, y, a.l2[1]);
    const double nyyy = fma(-m0, tA[5], s[C_OYYY]);
    const double hz = DIPOLE ? d2 * m1z : 0.0;
    a.l0 = fma(m0, -w, a.l0);
    a.l2[2] = fma(vx, z, a.l2[2]);
    const double c1 = DIPOLE ? fma(d2, ar, e1) : e1;
    a.l3[4] = fma(fzz, x, a.l3[4]);
    const double Vx = fma(qxz, z, fma(qxy, y, qxx * x));
    if (DIPOLE) a.l0 = fma(d1, ar, a.l0);
    const double e3xy = e3x * y;
    const double Vy = fma(qyz, z, fma(qyy, y, qxy * x));
    a.l2[3] += fma(vy, y, c1);
    const double S = fma(z, Vz, fma(y, Vy, x * Vx));
    a.l3[3] = fma(fyy, z, a.l3[3]);
    if (DIPOLE) a.l2[3] = fma(hy, y, a.l2[3]);
    a.l3[6] = fma(e3xy, z, a.l3[6]);
    const double pb = fma(y, y, -zz);
    if (DIPOLE) a.l2[1] = fma(hy, x, a.l2[1]);
    a.l2[4] = fma(vy, z, a.l2[4]);
    const double k1 = fma(d3, S, c1);
    const double u2 = d2 + d2;
    const double Qx = fma(nxyz, pyz, fma(nxxz, pxz, fma(nxxy, pxy, fma(nxyy, pb, nxxx * pa))));
    a.l3[0] = fma(fxx, y, a.l3[0]);
    a.l1[2] = fma(k1, z, a.l1[2]);
    a.l2[0] += fma(vx, x, c1);
    if (DIPOLE) a.l1[0] = fma(d1, m1x, a.l1[0]);
    a.l0b = fma(d2, S, a.l0b);
    const double nyzz = -(nxxy + nyyy);
    const double Qy = fma(nyyz, pyz, fma(nxyz, pxz, fma(nxyy, pxy, fma(nyyy, pb, nxxy * pa))));
    a.l3[1] = fma(fxx, z, a.l3[1]);
    const double Qz = fma(nyzz, pyz, fma(nxzz, pxz, fma(nxyz, pxy, fma(nyyz, pb, nxxz * pa))));
    const double C = fma(z, Qz, fma(y, Qy, x * Qx));
    a.l1[2] = fma(u2, Vz, a.l1[2]);
    a.l1[0] = fma(k1, x, a.l1[0]);
    if (DIPOLE) a.l2[4] = fma(hz, y, a.l2[4]);
    const double t4 = d3k7 * C;
    a.l1[1] = fma(k1, y, a.l1[1]);
    if (DIPOLE) a.l2[2] = fma(hz, x, a.l2[2]);
    a.l0 = fma(d3, C, a.l0);
    a.c[0] = fma(t4, x, a.c[0]);
    a.c[0] = fma(d3, Qx, a.c[0]);
    a.c[1] = fma(t4, y, a.c[1]);
    a.c[1] = fma(d3, Qy, a.c[1]);
    a.c[2] = fma(t4, z, a.c[2]);
    if (DIPOLE) a.l2[0] = fma(hx, x, a.l2[0]);
    a.c[2] = fma(d3, Qz, a.c[2]);
    a.l1[0] = fma(u2, Vx, a.l1[0]);
    a.l1[1] = fma(u2, Vy, a.l1[1]);
}

// Body of one ordered pair with the correction OFF, component form: the contractions
//   L0     += M D0 - M1.D1 + 1/2 M2:D2 - 1/6 M3:.D3
//   L1_i   += M D1_i - M1_j D2_ij + 1/2 M2_jk D3_ijk
//   L2_ij  += M D2_ij - M1_k D3_ijk            (xx xy xz yy yz)
//   L3_ijk += M D3_ijk                         (xxx xxy xxz xyy xyz yyy yyz)
// with the components of D generated one after the other (D2_ij = d1 d_ij + d2 R_i R_j, D3 likewise, zz / xzz / yzz from the
// traces) and every accumulation that uses a component written as a statement of its own; L0 alternates between two
// partial sums.  One statement per line, in an order found like the one of m2l_pair_folded (order_search): what counts is
// how often consecutive DFMAs share an operand slot (operand-reuse cache).
template <bool DIPOLE>
__device__ __forceinline__ void m2l_pair_components(Acc& a, const double x, const double y, const double z, const double w,
                                                     const double (&s)[16])
{
    const double w2 = w * w;
    const double d1 = w * w2;
    const double d2 = d1 * (-3.0 * w2);
    const double d3 = d2 * (-5.0 * w2);
    const double m0 = s[C_M0];
    const double m1x = s[C_M1X];
    const double m1y = s[C_M1Y];
    const double m1z = s[C_M1Z];
    const double qxx = s[C_QXX];
    const double qxy = s[C_QXY];
    const double qxz = s[C_QXZ];
    const double qyy = s[C_QYY];
    const double qyz = s[C_QYZ];
    const double oxxx = s[C_OXXX];
    const double oxxy = s[C_OXXY];
    const double oxxz = s[C_OXXZ];
    const double oxyy = s[C_OXYY];
    const double oxyz = s[C_OXYZ];
    const double oyyy = s[C_OYYY];
    const double oyyz = s[C_OYYZ];
    a.l0 = fma(m0, -w, a.l0);
    const double D1x = d1 * x;
    const double D1y = d1 * y;
    const double D1z = d1 * z;
    a.l1[0] = fma(m0, D1x, a.l1[0]);
    if (DIPOLE) a.l0b = fma(m1x, D1x, a.l0b);
    a.l1[1] = fma(m0, D1y, a.l1[1]);
    if (DIPOLE) a.l0 = fma(m1y, D1y, a.l0);
    a.l1[2] = fma(m0, D1z, a.l1[2]);
    if (DIPOLE) a.l0b = fma(m1z, D1z, a.l0b);
    const double ax = d2 * x;
    const double ay = d2 * y;
    const double az = d2 * z;
    const double Dxx = fma(ax, x, d1);
    const double Dyy = fma(ay, y, d1);
    const double Dzz = fma(az, z, d1);
    const double Dxy = ax * y;
    const double Dxz = ax * z;
    const double Dyz = ay * z;
    a.l2[0] = fma(m0, Dxx, a.l2[0]);
    if (DIPOLE) a.l1[0] = fma(m1x, Dxx, a.l1[0]);
    a.l0 = fma(qxx, Dxx, a.l0);
    a.l2[1] = fma(m0, Dxy, a.l2[1]);
    if (DIPOLE) a.l1[1] = fma(m1x, Dxy, a.l1[1]);
    if (DIPOLE) a.l1[0] = fma(m1y, Dxy, a.l1[0]);
    a.l0b = fma(qxy, Dxy, a.l0b);
    a.l2[2] = fma(m0, Dxz, a.l2[2]);
    if (DIPOLE) a.l1[2] = fma(m1x, Dxz, a.l1[2]);
    if (DIPOLE) a.l1[0] = fma(m1z, Dxz, a.l1[0]);
    a.l0 = fma(qxz, Dxz, a.l0);
    a.l2[3] = fma(m0, Dyy, a.l2[3]);
    if (DIPOLE) a.l1[1] = fma(m1y, Dyy, a.l1[1]);
    a.l0b = fma(qyy, Dyy, a.l0b);
    a.l2[4] = fma(m0, Dyz, a.l2[4]);
    if (DIPOLE) a.l1[2] = fma(m1y, Dyz, a.l1[2]);
    if (DIPOLE) a.l1[1] = fma(m1z, Dyz, a.l1[1]);
    a.l0 = fma(qyz, Dyz, a.l0);
    if (DIPOLE) a.l1[2] = fma(m1z, Dzz, a.l1[2]);
    const double bx = d3 * x;
    const double by = d3 * y;
    const double bxx = bx * x;
    const double bxy = bx * y;
    const double byy = by * y;
    const double ax3 = 3.0 * ax;
    const double ay3 = 3.0 * ay;
    const double Dxxx = fma(bxx, x, ax3);
    const double Dxxy = fma(bxx, y, ay);
    const double Dxxz = fma(bxx, z, az);
    a.l3[0] = fma(m0, Dxxx, a.l3[0]);
    if (DIPOLE) a.l2[0] = fma(m1x, Dxxx, a.l2[0]);
    a.l1[0] = fma(qxx, Dxxx, a.l1[0]);
    a.l0b = fma(oxxx, Dxxx, a.l0b);
    a.l3[1] = fma(m0, Dxxy, a.l3[1]);
    if (DIPOLE) a.l2[1] = fma(m1x, Dxxy, a.l2[1]);
    if (DIPOLE) a.l2[0] = fma(m1y, Dxxy, a.l2[0]);
    a.l1[1] = fma(qxx, Dxxy, a.l1[1]);
    a.l1[0] = fma(qxy, Dxxy, a.l1[0]);
    a.l0 = fma(oxxy, Dxxy, a.l0);
    a.l3[2] = fma(m0, Dxxz, a.l3[2]);
    if (DIPOLE) a.l2[2] = fma(m1x, Dxxz, a.l2[2]);
    if (DIPOLE) a.l2[0] = fma(m1z, Dxxz, a.l2[0]);
    a.l1[2] = fma(qxx, Dxxz, a.l1[2]);
    a.l1[0] = fma(qxz, Dxxz, a.l1[0]);
    a.l0b = fma(oxxz, Dxxz, a.l0b);
    const double Dxyy = fma(bxy, y, ax);
    const double Dxyz = bxy * z;
    a.l3[3] = fma(m0, Dxyy, a.l3[3]);
    if (DIPOLE) a.l2[3] = fma(m1x, Dxyy, a.l2[3]);
    if (DIPOLE) a.l2[1] = fma(m1y, Dxyy, a.l2[1]);
    a.l1[0] = fma(qyy, Dxyy, a.l1[0]);
    a.l1[1] = fma(qxy, Dxyy, a.l1[1]);
    a.l0 = fma(oxyy, Dxyy, a.l0);
    a.l3[4] = fma(m0, Dxyz, a.l3[4]);
    if (DIPOLE) a.l2[4] = fma(m1x, Dxyz, a.l2[4]);
    if (DIPOLE) a.l2[2] = fma(m1y, Dxyz, a.l2[2]);
    if (DIPOLE) a.l2[1] = fma(m1z, Dxyz, a.l2[1]);
    a.l1[0] = fma(qyz, Dxyz, a.l1[0]);
    a.l1[1] = fma(qxz, Dxyz, a.l1[1]);
    a.l1[2] = fma(qxy, Dxyz, a.l1[2]);
    a.l0b = fma(oxyz, Dxyz, a.l0b);
    const double Dyyy = fma(byy, y, ay3);
    const double Dyyz = fma(byy, z, az);
    a.l3[5] = fma(m0, Dyyy, a.l3[5]);
    if (DIPOLE) a.l2[3] = fma(m1y, Dyyy, a.l2[3]);
    a.l1[1] = fma(qyy, Dyyy, a.l1[1]);
    a.l0 = fma(oyyy, Dyyy, a.l0);
    a.l3[6] = fma(m0, Dyyz, a.l3[6]);
    if (DIPOLE) a.l2[4] = fma(m1y, Dyyz, a.l2[4]);
    if (DIPOLE) a.l2[3] = fma(m1z, Dyyz, a.l2[3]);
    a.l1[2] = fma(qyy, Dyyz, a.l1[2]);
    a.l1[1] = fma(qyz, Dyyz, a.l1[1]);
    a.l0b = fma(oyyz, Dyyz, a.l0b);
    const double Dxzz = -(Dxxx + Dxyy);
    const double Dyzz = -(Dxxy + Dyyy);
    if (DIPOLE) a.l2[2] = fma(m1z, Dxzz, a.l2[2]);
    a.l1[2] = fma(qxz, Dxzz, a.l1[2]);
    if (DIPOLE) a.l2[4] = fma(m1z, Dyzz, a.l2[4]);
    a.l1[2] = fma(qyz, Dyzz, a.l1[2]);
}

// Body of one ordered pair A <- B.  (x,y,z) = R = z_A - z_B, w = 1/|R|; s[0..15] staged source
// components; tA[0..6] = staged third moments of the target divided by its mass (correction only).
// DIPOLE = false leaves out the 27 terms with the source's dipole moment (and D2_zz, which only they need):
// the fast path for sources expanded about their centre of mass, chosen on the device (kernels.cuh).
template <bool CORR, bool DIPOLE>
__device__ __forceinline__ void m2l_pair(Acc& a, const double x, const double y, const double z, const double w,
                                         const double (&s)[16], const double (&tA)[7])
{
    if constexpr (CORR) m2l_pair_folded<DIPOLE>(a, x, y, z, w, s, tA);
    else                m2l_pair_components<DIPOLE>(a, x, y, z, w, s);
}

// Rebuild the 20 + 3 output coefficients from the accumulators.
template <bool CORR>
__device__ __forceinline__ void acc_finish(const Acc& a, const double (&tA)[7], double L[20], double C[3])
{
    L[0] = a.l0 + a.l0b;
#pragma unroll
    for (int i = 0; i < 3; ++i) {
        C[i] = CORR ? 3.0 * a.c[i] : 0.0;              // m2l_pair_folded accumulates a third of it
        L[1 + i] = CORR ? a.l1[i] + C[i] : a.l1[i];
    }
    double l2[5], l3[7];
#pragma unroll
    for (int i = 0; i < 5; ++i) l2[i] = a.l2[i];
    double xzz, yzz;
    if (CORR) {
        // m2l_pair_folded carries xxy xxz xyy yyz xzz yzz xyz; the repeated-index components follow from the traces
        l3[1] = a.l3[0]; l3[2] = a.l3[1]; l3[3] = a.l3[2]; l3[6] = a.l3[3]; l3[4] = a.l3[6];
        xzz = a.l3[4]; yzz = a.l3[5];
        l3[0] = -(l3[3] + xzz);                        // xxx = -(xyy + xzz)
        l3[5] = -(l3[1] + yzz);                        // yyy = -(xxy + yzz)
    } else {
#pragma unroll
        for (int i = 0; i < 7; ++i) l3[i] = a.l3[i];
        xzz = -(l3[0] + l3[3]);                        // xzz = -(xxx + xyy)
        yzz = -(l3[1] + l3[5]);                        // yzz = -(xxy + yyy)
    }
    if (CORR) {
        // the sources' octupoles entered L0 only through n = N'_B - M_B tA; the rest, sum_B M_B (tA :. D3(R_B)) =
        // tA :. L3, is added here, with tA taken to the reduced form that contracts with the 7 independent
        // components of the trace-free L3
        double t = 0.0;
        t = fma(fma(4.0, tA[0], 3.0 * tA[3]), l3[0], t);       // xxx
        t = fma(fma(6.0, tA[1], 3.0 * tA[5]), l3[1], t);       // xxy
        t = fma(fma(4.0, tA[2], tA[6]), l3[2], t);             // xxz
        t = fma(fma(6.0, tA[3], 3.0 * tA[0]), l3[3], t);       // xyy
        t = fma(6.0 * tA[4], l3[4], t);                        // xyz
        t = fma(fma(4.0, tA[5], 3.0 * tA[1]), l3[5], t);       // yyy
        t = fma(fma(4.0, tA[6], tA[2]), l3[6], t);             // yyz
        L[0] += t;
    }
    L[4] = l2[0]; L[5] = l2[1]; L[6] = l2[2]; L[7] = l2[3]; L[8] = l2[4];
    L[9] = -(l2[0] + l2[3]);                           // zz = -(xx + yy)
    L[10] = l3[0]; L[11] = l3[1]; L[12] = l3[2]; L[13] = l3[3]; L[14] = l3[4];
    L[15] = xzz;
    L[16] = l3[5]; L[17] = l3[6];
    L[18] = yzz;
    L[19] = -(l3[2] + l3[6]);                          // zzz = -(xxz + yyz)
}

}  // namespace octo
