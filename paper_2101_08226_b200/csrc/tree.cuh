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
// and the offset 0), an absent cell is all zeros.  The refined cells are written by m2m_kernel.  Only M0 ever changes from
// solve to solve: the zeros of raw and off, and of the cell's staged record S (the slab-fed kernel's source array), are
// written once, at octo_fmm_tree_create (tree_stage_init_kernel) -- per solve a cell that is not refined costs its mass in
// raw, in lm and in the first component pair of its staged record, 41 bytes instead of the 570 of writing and staging all
// 23 numbers.  lm (may be null): the masked masses [n^3] (m at leaves, 0 elsewhere) for the leaf kernel's staging.
__global__ void __launch_bounds__(256) tree_leaf_moments_kernel(const unsigned char* __restrict__ kind, const double* __restrict__ mass,
                                                                double* __restrict__ raw, double* __restrict__ lm,
                                                                double* __restrict__ S, int nx, int ny, long long ncell)
{
    const long long cell = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (cell >= ncell) return;
    const unsigned char kd = kind[cell];
    const double m = kd == KIND_LEAF ? mass[cell] : 0.0;
    if (lm) lm[cell] = m;
    if (kd == KIND_REFINED || !raw) return;
    raw[cell] = m;
    const int x = (int)(cell % nx);
    const long long r = cell / nx;
    const int y = (int)(r % ny);
    const long long z = r / ny;
    const long long plane = (long long)ny * nx;
    // (M0, -M1_x) of a point mass at the cell centre, as reduce_moments writes it
    if (S) reinterpret_cast<double2*>(S)[z * NPAIR * plane + (long long)y * nx + (x & 1) * (nx >> 1) + (x >> 1)] = make_double2(m, -0.0);
}

// Once per tree: the staged record of every cell as staging would write it for all-zero moments, with the cell's kind in the
// padding slot (0 absent, 1 leaf, 2 refined: what MODE_TREE reads beside a partner's moments).
__global__ void __launch_bounds__(256) tree_stage_init_kernel(const unsigned char* __restrict__ kind, double* __restrict__ S,
                                                              int nx, int ny, int nz, int corr)
{
    const long long cell = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (cell >= (long long)nx * ny * nz) return;
    const int x = (int)(cell % nx);
    const long long r = cell / nx;
    const int y = (int)(r % ny);
    const long long z = r / ny;
    double M[20], s[20];
#pragma unroll
    for (int c = 0; c < 20; ++c) M[c] = 0.0;
    reduce_moments(M, s, corr != 0);
    s[C_DX] = 0.0; s[C_DY] = 0.0; s[C_DZ] = 0.0;
    s[19] = (double)kind[cell];
    const long long plane = (long long)ny * nx;
    double2* dst = reinterpret_cast<double2*>(S) + z * NPAIR * plane + (long long)y * nx + (x & 1) * (nx >> 1) + (x >> 1);
#pragma unroll
    for (int c = 0; c < NPAIR; ++c) dst[(long long)c * plane] = make_double2(s[2 * c], s[2 * c + 1]);
}

// Per solve: the REFINED cells of a level (the sub-grids of `nodes`, 4 blocks of 128 threads each), staged as
// stage_multipole_kernel stages a cell -- moments reduced, dipole terms flagged, offsets -- with kind 2 in the padding slot.
__global__ void __launch_bounds__(128) tree_stage_refined_kernel(const double* __restrict__ mom, const double* __restrict__ com,
                                                                 double* __restrict__ S, int nx, int ny, int nz, double h,
                                                                 int* __restrict__ flags, int corr, const int* __restrict__ nodes)
{
    const int node = nodes[blockIdx.x >> 2];
    const int x = 8 * (node & 1023) + (threadIdx.x & 7), y = 8 * ((node >> 10) & 1023) + ((threadIdx.x >> 3) & 7),
              z = 8 * (node >> 20) + 2 * (blockIdx.x & 3) + (threadIdx.x >> 6);
    const long long ncell = (long long)nx * ny * nz;
    const long long cell = ((long long)z * ny + y) * nx + x;
    double M[20], s[20];
#pragma unroll
    for (int c = 0; c < 20; ++c) M[c] = mom[(long long)c * ncell + cell];
    reduce_moments(M, s, corr != 0);
    {
        const double lim = DIPOLE_TOL * fabs(M[0]) * h;
        if (fabs(M[1]) > lim || fabs(M[2]) > lim || fabs(M[3]) > lim) atomicOr(flags + 1, 2);
    }
#pragma unroll
    for (int c = 0; c < 3; ++c) s[C_DX + c] = com[(long long)c * ncell + cell];
    s[19] = (double)KIND_REFINED;
    const long long plane = (long long)ny * nx;
    double2* dst = reinterpret_cast<double2*>(S) + (long long)z * NPAIR * plane + (long long)y * nx + (x & 1) * (nx >> 1) + (x >> 1);
#pragma unroll
    for (int c = 0; c < NPAIR; ++c) dst[(long long)c * plane] = make_double2(s[2 * c], s[2 * c + 1]);
}

// L2L on a tree level stored as a box: what the fused epilogue of the brick kernel does when the levels run one after the
// other, as a pass of its own so that the multipole steps of ALL levels can run side by side and only this cheap chain is
// sequential.  For every existing cell: the correction is taken out of L1 and carried beside it, the parent's expansion,
// Taylor-shifted to the cell's expansion centre, and the parent's correction are added.
//   parent index = (index >> 1) + psh;   e = ((a,b,c) - 1/2) h + delta - delta_P
struct TreeL2LArgs {
    int n[3], pn[3], psh[3];
    double h;
    const unsigned char* kind;
    double* L; double* C; const double* off;             // this level: [20], [3], [3] x cells
    const double* pL; const double* pC; const double* poff;
    const int* nodes;                  // the refined sub-grids of the level (x | y << 10 | z << 20): 4 blocks of 128 threads each
};

__global__ void __launch_bounds__(128) tree_l2l_kernel(const TreeL2LArgs a)
{
    const int nx = a.n[0], ny = a.n[1], nz = a.n[2];
    const int node = a.nodes[blockIdx.x >> 2];
    const int i = 8 * (node & 1023) + (threadIdx.x & 7), j = 8 * ((node >> 10) & 1023) + ((threadIdx.x >> 3) & 7),
              k = 8 * (node >> 20) + 2 * (blockIdx.x & 3) + (threadIdx.x >> 6);
    if (i >= nx) return;
    const long long ncell = (long long)nx * ny * nz, cell = ((long long)k * ny + j) * nx + i;
    if (a.kind[cell] != KIND_REFINED) return;             // leaves take the parent's expansion in the leaf finish
    const long long pcell = (long long)a.pn[0] * a.pn[1] * a.pn[2];
    const long long P = ((long long)((k >> 1) + a.psh[2]) * a.pn[1] + ((j >> 1) + a.psh[1])) * a.pn[0] + ((i >> 1) + a.psh[0]);
    double e[3], Lp[20], sh[20], C[3];
    e[0] = ((double)(i & 1) - 0.5) * a.h + a.off[cell] - a.poff[P];
    e[1] = ((double)(j & 1) - 0.5) * a.h + a.off[ncell + cell] - a.poff[pcell + P];
    e[2] = ((double)(k & 1) - 0.5) * a.h + a.off[2 * ncell + cell] - a.poff[2 * pcell + P];
#pragma unroll
    for (int t = 0; t < 20; ++t) Lp[t] = a.pL[t * pcell + P];
#pragma unroll
    for (int c = 0; c < 3; ++c) C[c] = a.C[c * ncell + cell];
    taylor_shift<3>(Lp, e, sh);
#pragma unroll
    for (int t = 0; t < 20; ++t) {
        double v = a.L[t * ncell + cell];
        if (t >= 1 && t <= 3) v -= C[t - 1];
        a.L[t * ncell + cell] = v + sh[t];
    }
#pragma unroll
    for (int c = 0; c < 3; ++c) a.C[c * ncell + cell] = C[c] + a.pC[c * pcell + P];
}

struct TreeFinishArgs {
    int n[3];                       // extents of this level's arrays (a box of its lattice, multiples of 8)
    double h;                       // its cell width
    const unsigned char* kind;      // [nz][ny][nx]
    const unsigned char* nodeflag;  // [(nz/8)][(ny/8)][(nx/8)]
    double* out;                    // [4][cells]: in = leaf-leaf point-mass sums of the tensor-core kernel; out = (phi, g)
    const double* L;                // this level's own multipole step [20][cells], as stored by the brick kernel (correction
                                    // folded into L1); read at the leaves of sub-grids flagged NODE_OWN_L only, and there
    const unsigned char* brick_on;  // only in the 16 x 8 x 3 bricks the step ran on: brick_on[((j / TILE_Y) btx + i / TILE_X) btz + k / TILE_Z]
    int btx, btz;                   // (the others have no refined cell within the lists' reach: their part is exactly zero)
    const double* pL;               // parent level [20][pn cells], pC [3][..], poff [3][..]
    const double* pC;
    const double* poff;
    int pn[3];                      // extents of the parent arrays;  parent index = (index >> 1) + psh
    int psh[3];
    const unsigned char* kind_f;    // level below, or null: [fn cells];  child index = 2 * index + (a,b,c) + fsh
    const double* mass_f;           // its masked masses
    int fn[3];
    int fsh[3];
    const unsigned char* kind_c;    // level above (= the parent arrays' level), or null: [pn cells]
    const double* mass_c;
    unsigned long long* count;      // null, or counts[2] += cross-level pairs taken (ordered)
    double* phi_only;               // null, or (second right-hand side) [cells]: only the potential is wanted; out is then
                                    // read (the leaf-leaf sums) but not written
    const int* nodes;               // the sub-grids of the listed leaf tiles (x | y << 10 | z << 20): 4 blocks of 128 threads each;
                                    // the rest of the level's output was zero-filled before
};

// Leaf finish, one thread per cell of the level.  For a leaf A:
//   phi = [leaf-leaf sum] + expansion at its centre,  g = [leaf-leaf sum] - (L1 + correction), where the expansion is
//   the parent's, evaluated at the leaf centre, plus -- in sub-grids flagged NODE_OWN_L -- this level's own multipole step
//   (the refined cells of the Eq. 15 list);
//   + the children of the refined cells of its near field (NODE_OWN_L) and the coarser leaves in the near field of its
//   parent (NODE_COARSE_NBR), as point masses:  x_A - x_b = ((double)(2 i_A - i_b) + 0.5) * (h / 2) per axis, i the
//   index on the level's own LATTICE (the box shifts drop out of the difference: 2 i_A - i_b = 2 (A - B) - (a,b,c) for
//   the child (a,b,c) of B).
// Cells of the visited sub-grids that are not leaves get zeros (the rest of the level's output was zero-filled before the
// leaf-leaf sums).  The near-field offsets come from the constant bank (c_near).
__global__ void __launch_bounds__(128) tree_leaf_finish_kernel(const TreeFinishArgs a)
{
    const int nx = a.n[0], ny = a.n[1], nz = a.n[2];
    // a warp = 4 rows of one sub-grid: its flags, and with them every branch on them below, are the same for the warp
    const int node = a.nodes[blockIdx.x >> 2];
    const int i = 8 * (node & 1023) + (threadIdx.x & 7), j = 8 * ((node >> 10) & 1023) + ((threadIdx.x >> 3) & 7),
              k = 8 * (node >> 20) + 2 * (blockIdx.x & 3) + (threadIdx.x >> 6);
    if (i >= nx) return;
    const long long ncell = (long long)nx * ny * nz;
    const long long cell = ((long long)k * ny + j) * nx + i;
    if (a.kind[cell] != KIND_LEAF) {
        if (a.phi_only) { a.phi_only[cell] = 0.0; return; }
#pragma unroll
        for (int c = 0; c < 4; ++c) a.out[c * ncell + cell] = 0.0;
        return;
    }
    const unsigned char flag = a.nodeflag[((long long)(k >> 3) * (ny >> 3) + (j >> 3)) * (nx >> 3) + (i >> 3)];
    const int pi = (i >> 1) + a.psh[0], pj = (j >> 1) + a.psh[1], pk = (k >> 1) + a.psh[2];   // parent, in the parent arrays
    const long long pcell = (long long)a.pn[0] * a.pn[1] * a.pn[2];
    double v[4];
#pragma unroll
    for (int c = 0; c < 4; ++c) v[c] = a.out[c * ncell + cell];
    if ((flag & NODE_OWN_L) && a.brick_on[((j / TILE_Y) * a.btx + i / TILE_X) * a.btz + k / TILE_Z]) {
        // this level's own multipole step (refined partners of the Eq. 15 list), as the brick kernel stored it: the
        // correction folded into L1
        v[0] += a.L[cell];
#pragma unroll
        for (int c = 0; c < 3; ++c) v[1 + c] -= a.L[(1 + c) * ncell + cell];
    }
    {
        const long long P = ((long long)pk * a.pn[1] + pj) * a.pn[0] + pi;
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
    const int lane = threadIdx.x & 31;
    if ((flag & NODE_OWN_L) && a.kind_f) {
        // the children of the refined cells of the near field.  Kinds are constant over sub-grids and the warp's cells lie in
        // one: which of the 27 sub-grids around it are refined is read once (a lane each, one ballot); a partner's kind is
        // then a bit of that word -- no bounds test, no load per list entry
        unsigned char kd = KIND_ABSENT;
        {
            const int X = 8 * ((i >> 3) + lane % 3 - 1), Y = 8 * ((j >> 3) + (lane / 3) % 3 - 1), Z = 8 * ((k >> 3) + lane / 9 - 1);
            if (lane < 27 && X >= 0 && Y >= 0 && Z >= 0 && X < nx && Y < ny && Z < nz) kd = a.kind[((long long)Z * ny + Y) * nx + X];
        }
        const unsigned refined = __ballot_sync(0xffffffffu, kd == KIND_REFINED);
        const int cls = (i & 1) + 2 * (j & 1) + 4 * (k & 1);
        const double hf = 0.5 * a.h;
        double s[4] = {0.0, 0.0, 0.0, 0.0};
        for (int q = 0; q < c_near_count[cls]; ++q) {
            const char4 d = c_near[cls][q];
            const int bi = i + d.x, bj = j + d.y, bk = k + d.z;
            const int bit = ((((k & 7) + d.z) >> 3) + 1) * 9 + ((((j & 7) + d.y) >> 3) + 1) * 3 + ((((i & 7) + d.x) >> 3) + 1);
            if (!((refined >> bit) & 1u)) continue;
#pragma unroll
            for (int c = 0; c < 8; ++c) {
                const int ax = c & 1, ay = (c >> 1) & 1, az = c >> 2;
                const int ci = 2 * bi + ax + a.fsh[0], cj = 2 * bj + ay + a.fsh[1], ck = 2 * bk + az + a.fsh[2];   // in the fine arrays
                const double m = a.mass_f[((long long)ck * a.fn[1] + cj) * a.fn[0] + ci];
                const double Rx = ((double)(-2 * d.x - ax) + 0.5) * hf, Ry = ((double)(-2 * d.y - ay) + 0.5) * hf,
                             Rz = ((double)(-2 * d.z - az) + 0.5) * hf;
                const double w = rsqrt_fast(Rx * Rx + Ry * Ry + Rz * Rz), mw = -m * w, w3 = mw * (w * w);   // 1/r to < 1 ulp (m2l_math.cuh)
                s[0] += mw; s[1] += w3 * Rx; s[2] += w3 * Ry; s[3] += w3 * Rz;
                ++taken;
            }
        }
#pragma unroll
        for (int c = 0; c < 4; ++c) v[c] += s[c];
    }
    if ((flag & NODE_COARSE_NBR) && a.kind_c) {
        // the coarser leaves in the near field of the parent (the parents of a sub-grid's cells lie in one sub-grid of the
        // level above: the same word of 27 kinds, there)
        unsigned char kd = KIND_ABSENT;
        {
            const int X = 8 * ((pi >> 3) + lane % 3 - 1), Y = 8 * ((pj >> 3) + (lane / 3) % 3 - 1), Z = 8 * ((pk >> 3) + lane / 9 - 1);
            if (lane < 27 && X >= 0 && Y >= 0 && Z >= 0 && X < a.pn[0] && Y < a.pn[1] && Z < a.pn[2])
                kd = a.kind_c[((long long)Z * a.pn[1] + Y) * a.pn[0] + X];
        }
        const unsigned coarse_leaf = __ballot_sync(0xffffffffu, kd == KIND_LEAF);
        const int cls = (pi & 1) + 2 * (pj & 1) + 4 * (pk & 1);       // psh is even: the parity of the lattice index
        const double hf = a.h;                       // this level is the fine one of the pair
        double s[4] = {0.0, 0.0, 0.0, 0.0};
        for (int q = 0; q < c_near_count[cls]; ++q) {
            const char4 d = c_near[cls][q];
            const int ai = pi + d.x, aj = pj + d.y, ak = pk + d.z;
            const int bit = ((((pk & 7) + d.z) >> 3) + 1) * 9 + ((((pj & 7) + d.y) >> 3) + 1) * 3 + ((((pi & 7) + d.x) >> 3) + 1);
            if (!((coarse_leaf >> bit) & 1u)) continue;
            const long long A = ((long long)ak * a.pn[1] + aj) * a.pn[0] + ai;
            const double m = a.mass_c[A];
            // x_b - x_A = -(x_A - x_b),  2 i_A - i_b = 2 (parent + d) - (2 parent + (a,b,c)) = 2 d - (a,b,c)
            const double Rx = -(((double)(2 * d.x - (i & 1)) + 0.5) * hf), Ry = -(((double)(2 * d.y - (j & 1)) + 0.5) * hf),
                         Rz = -(((double)(2 * d.z - (k & 1)) + 0.5) * hf);
            const double w = rsqrt_fast(Rx * Rx + Ry * Ry + Rz * Rz), mw = -m * w, w3 = mw * (w * w);
            s[0] += mw; s[1] += w3 * Rx; s[2] += w3 * Ry; s[3] += w3 * Rz;
            ++taken;
        }
#pragma unroll
        for (int c = 0; c < 4; ++c) v[c] += s[c];
    }
    if (a.phi_only) {
        a.phi_only[cell] = v[0];
    } else {
#pragma unroll
        for (int c = 0; c < 4; ++c) a.out[c * ncell + cell] = v[c];
    }
    if (a.count && taken) atomicAdd(a.count + 2, taken);
}

// Pair counter of one level, for the bit-exact check of the pair set against the oracle: counts[0] += ordered pairs of the
// multipole step (both exist, on the Eq. 15 list, not two leaves), counts[1] += leaf-leaf point-mass pairs (leaf-level list).
// The Eq. 15 list is in the constant bank as 8 x (dx, dy, dz) of c_entries (a multipole list), the near field as c_near.
__global__ void __launch_bounds__(128) tree_count_kernel(const unsigned char* __restrict__ kind, int nx, int ny, int nz,
                                                         unsigned long long* __restrict__ counts)
{
    const int i = blockIdx.x * blockDim.x + threadIdx.x, j = blockIdx.y, k = blockIdx.z;
    unsigned long long m2l = 0, p2p = 0;
    if (i < nx) {
        const unsigned char ka = kind[((long long)k * ny + j) * nx + i];
        if (ka != KIND_ABSENT) {
            const int cls = (i & 1) + 2 * (j & 1) + 4 * (k & 1);
            const int s_end = c_begin[cls][2 * REACH_MAX + 1];
            for (int s = c_begin[cls][0]; s < s_end; ++s) {
                const StEntry e = c_entries[cls * MAX_LIST + s];
                const int bi = i + (e.dx >> 3), bj = j + (e.dy >> 3), bk = k + (e.dz >> 3);    // multipole lists hold 8 d
                if (bi < 0 || bj < 0 || bk < 0 || bi >= nx || bj >= ny || bk >= nz) continue;
                const unsigned char kb = kind[((long long)bk * ny + bj) * nx + bi];
                if (kb == KIND_ABSENT) continue;
                if (ka == KIND_LEAF && kb == KIND_LEAF) ++p2p; else ++m2l;
            }
            if (ka == KIND_LEAF)
                for (int q = 0; q < c_near_count[cls]; ++q) {
                    const char4 d = c_near[cls][q];
                    const int bi = i + d.x, bj = j + d.y, bk = k + d.z;
                    if (bi < 0 || bj < 0 || bk < 0 || bi >= nx || bj >= ny || bk >= nz) continue;
                    if (kind[((long long)bk * ny + bj) * nx + bi] == KIND_LEAF) ++p2p;
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
