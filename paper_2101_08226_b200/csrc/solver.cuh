// solver.cuh -- the other passes of a complete uniform-grid solve, sm_100a.
//
// "The multipoles of each cell are composed of the multipoles of its child cells ... The expansion of each
// cell is composed of the expansion due to its interactions with other cells at the same level, and the
// expansion of its parent cell".  The same-level interactions are the hot path
// (kernels.cuh); here are the upward pass (M2M), the downward pass (L2L) and the leaf evaluation.
// All three are HBM-bound, one thread per cell, SoA arrays [comp][z][y][x], positions kept relative
// to the parent's geometric centre.  Formulas: DESIGN.md section 12.
#pragma once

#include <cuda_runtime.h>

#include "taylor.cuh"

namespace octo {

// ------------------------------------------------------------------------------------------
// M2M: parent multipoles (order 3, raw moments about the parent's centre of mass) from its 8
// children.  LEAF: the children are point masses at their cell centres (cm = mass [nz][ny][nx],
// coff unused); otherwise cm = [20][child grid], coff = [3][child grid].
//   rel_c = ((a,b,c) - 1/2) hc + delta_c;   delta_P = sum_c (M_c rel_c + M1_c) / sum_c M_c  (0 if the mass is 0)
//   d = rel_c - delta_P;  M1' = M1 + M d;  M2'_ij = M2_ij + M1_i d_j + M1_j d_i + M d_i d_j;
//   M3'_ijk = M3_ijk + (M2_ij d_k + M2_ik d_j + M2_jk d_i) + (M1_i d_j d_k + M1_j d_i d_k + M1_k d_i d_j) + M d_i d_j d_k
// GIVEN (second right-hand side, L81-83: d(rho)/dt expanded about the centres of rho): delta_P is read from poff
// instead of being computed and written; coff are then the children's centres from the first right-hand side.
// ------------------------------------------------------------------------------------------
// Child arrays stored as a BOX of their lattice (levels of the adaptive tree): cbox = extents of the child arrays and the
// (even) shift of the child index, child = 2 * parent + (a,b,c) + sh; children outside the box do not exist (zero mass).
// The uniform solve passes a null box: the child arrays are exactly twice the parent's.
struct ChildBox { int n[3]; int sh[3]; const unsigned char* pkind; const int* nodes = nullptr; };
// nodes (may be null): the refined 8^3 sub-grids of the parent level, x | y << 10 | z << 20 in sub-grid units: the grid is then
// 4 blocks of 128 threads per listed sub-grid instead of one thread per cell of the box.    pkind (may be null): kind of every parent cell; only
                                                                        // the refined ones (2) are built from children

template <bool LEAF, bool GIVEN = false, bool BOXED = false>
__global__ void __launch_bounds__(128) m2m_kernel(const double* __restrict__ cm, const double* __restrict__ coff,
                                                  double* __restrict__ pm, double* __restrict__ poff, int pnx, int pny, int pnz,
                                                  double hc, const ChildBox cb = ChildBox())
{
    // grid = (ceil(pnx / blockDim.x), pny, pnz): no integer divisions
    const long long pcell = (long long)pnx * pny * pnz;
    int I = blockIdx.x * blockDim.x + threadIdx.x, J = blockIdx.y, K = blockIdx.z;
    if (BOXED && cb.nodes) {                               // only the refined sub-grids: every lane of every warp has work
        const int node = cb.nodes[blockIdx.x >> 2];
        I = 8 * (node & 1023) + (threadIdx.x & 7);
        J = 8 * ((node >> 10) & 1023) + ((threadIdx.x >> 3) & 7);
        K = 8 * (node >> 20) + 2 * (blockIdx.x & 3) + (threadIdx.x >> 6);
    }
    if (I >= pnx) return;
    const long long P = ((long long)K * pny + J) * pnx + I;
    if (BOXED && cb.pkind && cb.pkind[P] != 2) return;      // a leaf or absent parent: tree_leaf_moments_kernel writes it
    const int cnx = BOXED ? cb.n[0] : 2 * pnx, cny = BOXED ? cb.n[1] : 2 * pny, cnz = BOXED ? cb.n[2] : 2 * pnz;
    const long long ccell = (long long)cnx * cny * cnz;
    long long cell[8];
    double rel[8][3], m0s[8];
    double mass = 0.0, com[3] = {0.0, 0.0, 0.0};
    // all eight children are inside the child box or none is (the shift is even and so are the extents)
    const int cx0 = 2 * I + (BOXED ? cb.sh[0] : 0), cy0 = 2 * J + (BOXED ? cb.sh[1] : 0), cz0 = 2 * K + (BOXED ? cb.sh[2] : 0);
    const bool inside = !BOXED || (cx0 >= 0 && cy0 >= 0 && cz0 >= 0 && cx0 < cnx && cy0 < cny && cz0 < cnz);
#pragma unroll
    for (int c = 0; c < 8; ++c) {
        const int a[3] = {c & 1, (c >> 1) & 1, (c >> 2) & 1};
        cell[c] = inside ? ((long long)(cz0 + a[2]) * cny + (cy0 + a[1])) * cnx + (cx0 + a[0]) : (long long)a[0];
        double m0;
        if (LEAF) {          // the two x-children are one aligned double2 (cm is 16-byte aligned, cnx is even)
            const double2 pair = *reinterpret_cast<const double2*>(cm + (cell[c] - a[0]));
            m0 = a[0] ? pair.y : pair.x;
        } else {
            m0 = cm[cell[c]];
        }
        if (BOXED && !inside) m0 = 0.0;
        m0s[c] = m0;
#pragma unroll
        for (int i = 0; i < 3; ++i) {
            const bool none = LEAF || (BOXED && !inside);
            rel[c][i] = ((double)a[i] - 0.5) * hc + (none ? 0.0 : coff[i * ccell + cell[c]]);
            com[i] += m0 * rel[c][i] + (none ? 0.0 : cm[(1 + i) * ccell + cell[c]]);
        }
        mass += m0;
    }
    double dP[3] = {0.0, 0.0, 0.0};
    if (GIVEN) {
#pragma unroll
        for (int i = 0; i < 3; ++i) dP[i] = poff[i * pcell + P];
    } else if (mass != 0.0) {
#pragma unroll
        for (int i = 0; i < 3; ++i) dP[i] = com[i] / mass;
    }
    double S[20];
#pragma unroll
    for (int t = 0; t < 20; ++t) S[t] = 0.0;
    S[0] = mass;
#pragma unroll
    for (int c = 0; c < 8; ++c) {
        double M[20];
        M[0] = m0s[c];
#pragma unroll
        for (int t = 1; t < 20; ++t) M[t] = (LEAF || (BOXED && !inside)) ? 0.0 : cm[t * ccell + cell[c]];
        double d[3];
#pragma unroll
        for (int i = 0; i < 3; ++i) d[i] = rel[c][i] - dP[i];
#pragma unroll
        for (int i = 0; i < 3; ++i) S[1 + i] += M[1 + i] + M[0] * d[i];
#pragma unroll
        for (int i = 0; i < 3; ++i)
#pragma unroll
            for (int j = i; j < 3; ++j)
                S[4 + u2(i, j)] += M[4 + u2(i, j)] + M[1 + i] * d[j] + M[1 + j] * d[i] + M[0] * d[i] * d[j];
#pragma unroll
        for (int i = 0; i < 3; ++i)
#pragma unroll
            for (int j = i; j < 3; ++j)
#pragma unroll
                for (int k = j; k < 3; ++k)
                    S[10 + u3(i, j, k)] += M[10 + u3(i, j, k)] + M[4 + u2(i, j)] * d[k] + M[4 + u2(i, k)] * d[j] +
                                           M[4 + u2(j, k)] * d[i] + M[1 + i] * d[j] * d[k] + M[1 + j] * d[i] * d[k] +
                                           M[1 + k] * d[i] * d[j] + M[0] * d[i] * d[j] * d[k];
    }
#pragma unroll
    for (int t = 0; t < 20; ++t) pm[t * pcell + P] = S[t];
    if (!GIVEN) {
#pragma unroll
        for (int i = 0; i < 3; ++i) poff[i * pcell + P] = dP[i];
    }
}

// ------------------------------------------------------------------------------------------
// L2L: cL = (cL with the correction taken out of L1) + parent expansion shifted to the child's
// centre; cC += parent correction (a uniform acceleration, handed down unchanged).
// HAS_PARENT = false (coarsest level): only the un-folding  L1 -= C.
//   e = ((a,b,c) - 1/2) hc + delta_c - delta_P
// ------------------------------------------------------------------------------------------
template <bool HAS_PARENT>
__global__ void __launch_bounds__(128) l2l_kernel(double* __restrict__ cL, double* __restrict__ cC, const double* __restrict__ coff,
                                                  const double* __restrict__ pL, const double* __restrict__ pC,
                                                  const double* __restrict__ poff, int cnx, int cny, int cnz, double hc)
{
    // grid = (ceil(cnx / blockDim.x), cny, cnz)
    const long long ccell = (long long)cnx * cny * cnz;
    const int i = blockIdx.x * blockDim.x + threadIdx.x, j = blockIdx.y, k = blockIdx.z;
    if (i >= cnx) return;
    const long long cell = ((long long)k * cny + j) * cnx + i;
    double C[3];
#pragma unroll
    for (int c = 0; c < 3; ++c) C[c] = cC[c * ccell + cell];
    if (!HAS_PARENT) {
#pragma unroll
        for (int c = 0; c < 3; ++c) cL[(1 + c) * ccell + cell] -= C[c];
        return;
    }
    const int pnx = cnx / 2, pny = cny / 2;
    const long long pcell = ccell / 8;
    const long long P = ((long long)(k / 2) * pny + (j / 2)) * pnx + (i / 2);
    const int a[3] = {i & 1, j & 1, k & 1};
    double e[3], L[20], sh[20];
#pragma unroll
    for (int c = 0; c < 3; ++c) e[c] = ((double)a[c] - 0.5) * hc + coff[c * ccell + cell] - poff[c * pcell + P];
#pragma unroll
    for (int t = 0; t < 20; ++t) L[t] = pL[t * pcell + P];
    taylor_shift<3>(L, e, sh);
#pragma unroll
    for (int t = 0; t < 20; ++t) {
        double v = cL[t * ccell + cell];
        if (t >= 1 && t <= 3) v -= C[t - 1];
        cL[t * ccell + cell] = v + sh[t];
    }
#pragma unroll
    for (int c = 0; c < 3; ++c) cC[c * ccell + cell] = C[c] + pC[c * pcell + P];
}

// ------------------------------------------------------------------------------------------
// Leaf evaluation: out = (phi, g) of the leaf-level monopole sum; add the parent's expansion
// evaluated at the leaf's cell centre:  phi += L0(e),  g -= L1(e) + correction,  e = ((a,b,c) - 1/2) h - delta_P.
// One thread per PARENT (grid = (ceil(pnx / blockDim.x), pny, pnz)): the parent's 26 numbers are read once
// and its 8 leaves are updated as four double2 (x-pairs), so every access of a warp is contiguous.
// out must be 16-byte aligned.  PHI_ONLY (second right-hand side): out = [nz][ny][nx], only the potential row.
// ------------------------------------------------------------------------------------------
template <bool PHI_ONLY = false>
__global__ void __launch_bounds__(128) leaf_eval_kernel(double* __restrict__ out, const double* __restrict__ pL,
                                                        const double* __restrict__ pC, const double* __restrict__ poff, int nx,
                                                        int ny, int nz, double h)
{
    const int pnx = nx / 2, pny = ny / 2;
    const int I = blockIdx.x * blockDim.x + threadIdx.x, J = blockIdx.y, K = blockIdx.z;
    if (I >= pnx) return;
    const long long ncell = (long long)nx * ny * nz, pcell = ncell / 8;
    const long long P = ((long long)K * pny + J) * pnx + I;
    double L[20], C[3], dP[3];
#pragma unroll
    for (int t = 0; t < 20; ++t) L[t] = pL[t * pcell + P];
#pragma unroll
    for (int c = 0; c < 3; ++c) { C[c] = pC[c * pcell + P]; dP[c] = poff[c * pcell + P]; }
#pragma unroll
    for (int cz = 0; cz < 2; ++cz)
#pragma unroll
        for (int cy = 0; cy < 2; ++cy) {
            const long long row = ((long long)(2 * K + cz) * ny + (2 * J + cy)) * nx + 2 * I;     // even: 16-byte aligned
            double sh0[20], sh1[20];
            const double e0[3] = {-0.5 * h - dP[0], ((double)cy - 0.5) * h - dP[1], ((double)cz - 0.5) * h - dP[2]};
            const double e1[3] = {0.5 * h - dP[0], e0[1], e0[2]};
            taylor_shift<1>(L, e0, sh0);
            taylor_shift<1>(L, e1, sh1);
            double2* o = reinterpret_cast<double2*>(out + row);
            double2 v = *o;
            v.x += sh0[0]; v.y += sh1[0];
            *o = v;
            if constexpr (!PHI_ONLY) {
#pragma unroll
                for (int c = 0; c < 3; ++c) {
                    double2* g = reinterpret_cast<double2*>(out + (1 + c) * ncell + row);
                    double2 w = *g;
                    w.x -= sh0[1 + c] + C[c]; w.y -= sh1[1 + c] + C[c];
                    *g = w;
                }
            }
        }
}

}  // namespace octo
