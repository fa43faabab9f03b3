// tree.cuh -- kernels of the gravity solve on an ADAPTIVE oct-tree of 8^3 sub-grids, sm_100a.
//
// PAPER.md L125 ("The FMM adapts naturally to an oct-tree based adaptive mesh refinement"), L287-291 (a node is fully
// refined or a leaf; proper nesting: a refinement boundary involves exactly two levels).  The paper does not describe the
// gravity side of such a boundary; reading R9 (section 12c) is the symmetric dual descent of the rule of L135:
// a pair that is well separated (parents not) interacts on its level with the general pair formula, whatever the kinds;
// a pair that is not is left to the children; two leaves meet as point masses; a leaf A and a refined B that are not
// well separated: A meets the eight CHILDREN of B (leaves one level down) as point masses, in both directions.
//
// A level is a dense [n][n][n] lattice with kind[cell] = 0 absent, 1 leaf, 2 refined (constant over 8^3 sub-grids).
// The heavy steps run on the kernels of kernels.cuh restricted to the bricks / tiles that have work (tile lists):
// m2l_staged_kernel<., FUSE_L2L, MODE_TREE> for the same-level multipole step and p2p_monopole_dmma_kernel for the
// leaf-leaf point-mass sums.  Here: the moments of the non-refined cells, and the leaf finish -- expansion at the leaf
// centre plus the point-mass pairs across a refinement boundary -- and the pair counter for the bit-exact check.
#pragma once

#include <cuda_runtime.h>

#include "kernels.cuh"
#include "taylor.cuh"

namespace octo {

constexpr unsigned char KIND_ABSENT = 0, KIND_LEAF = 1, KIND_REFINED = 2;
// per sub-grid flags, computed on the host at create()
constexpr unsigned char NODE_OWN_L = 1;          // leaf sub-grid with a refined sub-grid among its 26 neighbours: its cells take part in
                                                 // the level's multipole step (refined partners) and may have refined near-field cells
constexpr unsigned char NODE_COARSE_NBR = 2;     // the parent sub-grid has a LEAF sub-grid among its 26 neighbours one level up

// Moments of the cells that are not refined: a leaf is the point mass at its geometric centre (M0 = m, everything else
// and the offset 0), an absent cell is all zeros.  The refined cells were written by m2m_kernel before.  lm (may be
// null): the masked masses [n^3] (m at leaves, 0 elsewhere) for the leaf kernel's staging.
__global__ void __launch_bounds__(256) tree_leaf_moments_kernel(const unsigned char* __restrict__ kind, const double* __restrict__ mass,
                                                                double* __restrict__ raw, double* __restrict__ off,
                                                                double* __restrict__ lm, long long ncell)
{
    const long long cell = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (cell >= ncell) return;
    const unsigned char kd = kind[cell];
    const double m = kd == KIND_LEAF ? mass[cell] : 0.0;
    if (lm) lm[cell] = m;
    if (kd == KIND_REFINED || !raw) return;
    raw[cell] = m;
#pragma unroll
    for (int t = 1; t < 20; ++t) raw[t * ncell + cell] = 0.0;
#pragma unroll
    for (int c = 0; c < 3; ++c) off[c * ncell + cell] = 0.0;
}

struct TreeFinishArgs {
    int n;                          // cells per axis of this level
    double h;                       // its cell width
    const unsigned char* kind;      // [n^3]
    const unsigned char* nodeflag;  // [(n/8)^3]
    const double* lm;               // masked masses of this level (not used here; kept for symmetry)
    double* out;                    // [4][n^3]: in = leaf-leaf point-mass sums of the tensor-core kernel; out = (phi, g)
    const double* L;                // this level's finished expansions [20][n^3] (correction beside, parent's part included)
    const double* C;                // [3][n^3]
    const double* pL;               // parent level [20][(n/2)^3], pC [3][..], poff [3][..]
    const double* pC;
    const double* poff;
    const unsigned char* kind_f;    // level below: [(2n)^3] or null
    const double* mass_f;           // its masked masses
    const unsigned char* kind_c;    // level above: [(n/2)^3] or null
    const double* mass_c;
    unsigned long long* count;      // null, or counts[2] += cross-level pairs taken (ordered)
};

// Leaf finish, one thread per cell of the level.  For a leaf A:
//   phi = [leaf-leaf sum] + expansion at its centre,  g = [leaf-leaf sum] - (L1 + correction), where the expansion is
//   this level's own L (sub-grids flagged NODE_OWN_L: Eq. 15 partners that are refined + the parent's shifted expansion,
//   already added by the fused L2L epilogue) or else the parent's expansion evaluated at the leaf centre;
//   + the children of the refined cells of its near field (NODE_OWN_L) and the coarser leaves in the near field of its
//   parent (NODE_COARSE_NBR), as point masses:  x_A - x_b = ((double)(2 i_A - i_b) + 0.5) * (h / 2) per axis.
// Cells that are not leaves get zeros.  The near-field offsets come from the constant bank (c_near).
__global__ void __launch_bounds__(128) tree_leaf_finish_kernel(const TreeFinishArgs a)
{
    const int n = a.n;
    const int i = blockIdx.x * blockDim.x + threadIdx.x, j = blockIdx.y, k = blockIdx.z;
    if (i >= n) return;
    const long long ncell = (long long)n * n * n;
    const long long cell = ((long long)k * n + j) * n + i;
    if (a.kind[cell] != KIND_LEAF) {
#pragma unroll
        for (int c = 0; c < 4; ++c) a.out[c * ncell + cell] = 0.0;
        return;
    }
    const int nn = n >> 3;
    const unsigned char flag = a.nodeflag[((long long)(k >> 3) * nn + (j >> 3)) * nn + (i >> 3)];
    double v[4];
#pragma unroll
    for (int c = 0; c < 4; ++c) v[c] = a.out[c * ncell + cell];
    if (flag & NODE_OWN_L) {
        v[0] += a.L[cell];
#pragma unroll
        for (int c = 0; c < 3; ++c) v[1 + c] -= a.L[(1 + c) * ncell + cell] + a.C[c * ncell + cell];
    } else {
        const int pn = n >> 1;
        const long long pcell = ncell >> 3;
        const long long P = ((long long)(k >> 1) * pn + (j >> 1)) * pn + (i >> 1);
        double Lp[20], sh[20], e[3];
#pragma unroll
        for (int t = 0; t < 20; ++t) Lp[t] = a.pL[t * pcell + P];
        e[0] = ((double)(i & 1) - 0.5) * a.h - a.poff[P];
        e[1] = ((double)(j & 1) - 0.5) * a.h - a.poff[pcell + P];
        e[2] = ((double)(k & 1) - 0.5) * a.h - a.poff[2 * pcell + P];
        taylor_shift<1>(Lp, e, sh);
        v[0] += sh[0];
#pragma unroll
        for (int c = 0; c < 3; ++c) v[1 + c] -= sh[1 + c] + a.pC[c * pcell + P];
    }
    unsigned long long taken = 0;
    if ((flag & NODE_OWN_L) && a.kind_f) {
        // the children of the refined cells of the near field
        const int cls = (i & 1) + 2 * (j & 1) + 4 * (k & 1);
        const int fn = 2 * n;
        const double hf = 0.5 * a.h;
        double s[4] = {0.0, 0.0, 0.0, 0.0};
        for (int q = 0; q < c_near_count[cls]; ++q) {
            const char4 d = c_near[cls][q];
            const int bi = i + d.x, bj = j + d.y, bk = k + d.z;
            if (bi < 0 || bj < 0 || bk < 0 || bi >= n || bj >= n || bk >= n) continue;
            if (a.kind[((long long)bk * n + bj) * n + bi] != KIND_REFINED) continue;
#pragma unroll
            for (int c = 0; c < 8; ++c) {
                const int ci = 2 * bi + (c & 1), cj = 2 * bj + ((c >> 1) & 1), ck = 2 * bk + (c >> 2);
                const double m = a.mass_f[((long long)ck * fn + cj) * fn + ci];
                const double Rx = ((double)(2 * i - ci) + 0.5) * hf, Ry = ((double)(2 * j - cj) + 0.5) * hf,
                             Rz = ((double)(2 * k - ck) + 0.5) * hf;
                const double r2 = Rx * Rx + Ry * Ry + Rz * Rz, r = sqrt(r2), w3 = -m / (r2 * r);
                s[0] += -m / r; s[1] += w3 * Rx; s[2] += w3 * Ry; s[3] += w3 * Rz;
                ++taken;
            }
        }
#pragma unroll
        for (int c = 0; c < 4; ++c) v[c] += s[c];
    }
    if ((flag & NODE_COARSE_NBR) && a.kind_c) {
        // the coarser leaves in the near field of the parent
        const int pi = i >> 1, pj = j >> 1, pk = k >> 1, pn = n >> 1;
        const int cls = (pi & 1) + 2 * (pj & 1) + 4 * (pk & 1);
        const double hf = a.h;                       // this level is the fine one of the pair
        double s[4] = {0.0, 0.0, 0.0, 0.0};
        for (int q = 0; q < c_near_count[cls]; ++q) {
            const char4 d = c_near[cls][q];
            const int ai = pi + d.x, aj = pj + d.y, ak = pk + d.z;
            if (ai < 0 || aj < 0 || ak < 0 || ai >= pn || aj >= pn || ak >= pn) continue;
            const long long A = ((long long)ak * pn + aj) * pn + ai;
            if (a.kind_c[A] != KIND_LEAF) continue;
            const double m = a.mass_c[A];
            const double Rx = -(((double)(2 * ai - i) + 0.5) * hf), Ry = -(((double)(2 * aj - j) + 0.5) * hf),
                         Rz = -(((double)(2 * ak - k) + 0.5) * hf);
            const double r2 = Rx * Rx + Ry * Ry + Rz * Rz, r = sqrt(r2), w3 = -m / (r2 * r);
            s[0] += -m / r; s[1] += w3 * Rx; s[2] += w3 * Ry; s[3] += w3 * Rz;
            ++taken;
        }
#pragma unroll
        for (int c = 0; c < 4; ++c) v[c] += s[c];
    }
#pragma unroll
    for (int c = 0; c < 4; ++c) a.out[c * ncell + cell] = v[c];
    if (a.count && taken) atomicAdd(a.count + 2, taken);
}

// Pair counter of one level, for the bit-exact check of the pair set against the oracle: counts[0] += ordered pairs of the
// multipole step (both exist, on the Eq. 15 list, not two leaves), counts[1] += leaf-leaf point-mass pairs (leaf-level list).
// The Eq. 15 list is in the constant bank as (dx, dy, dz) of c_entries, the near field as c_near.
__global__ void __launch_bounds__(128) tree_count_kernel(const unsigned char* __restrict__ kind, int n, unsigned long long* __restrict__ counts)
{
    const int i = blockIdx.x * blockDim.x + threadIdx.x, j = blockIdx.y, k = blockIdx.z;
    unsigned long long m2l = 0, p2p = 0;
    if (i < n) {
        const unsigned char ka = kind[((long long)k * n + j) * n + i];
        if (ka != KIND_ABSENT) {
            const int cls = (i & 1) + 2 * (j & 1) + 4 * (k & 1);
            const int s_end = c_begin[cls][2 * REACH_MAX + 1];
            for (int s = c_begin[cls][0]; s < s_end; ++s) {
                const StEntry e = c_entries[cls * MAX_LIST + s];
                const int bi = i + e.dx, bj = j + e.dy, bk = k + e.dz;
                if (bi < 0 || bj < 0 || bk < 0 || bi >= n || bj >= n || bk >= n) continue;
                const unsigned char kb = kind[((long long)bk * n + bj) * n + bi];
                if (kb == KIND_ABSENT) continue;
                if (ka == KIND_LEAF && kb == KIND_LEAF) ++p2p; else ++m2l;
            }
            if (ka == KIND_LEAF)
                for (int q = 0; q < c_near_count[cls]; ++q) {
                    const char4 d = c_near[cls][q];
                    const int bi = i + d.x, bj = j + d.y, bk = k + d.z;
                    if (bi < 0 || bj < 0 || bk < 0 || bi >= n || bj >= n || bk >= n) continue;
                    if (kind[((long long)bk * n + bj) * n + bi] == KIND_LEAF) ++p2p;
                }
        }
    }
    for (int d = 16; d > 0; d >>= 1) {
        m2l += __shfl_xor_sync(0xffffffffu, m2l, d);
        p2p += __shfl_xor_sync(0xffffffffu, p2p, d);
    }
    if ((threadIdx.x & 31) == 0) {
        if (m2l) atomicAdd(counts, m2l);
        if (p2p) atomicAdd(counts + 1, p2p);
    }
}

}  // namespace octo
