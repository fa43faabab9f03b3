// kernels.cuh -- sm_100a kernels of the FMM cell-to-cell interaction step.
//
//   stage_multipole_kernel   a2: raw moments -> staged layout in the workspace
//   m2l_staged_kernel        a3/a4/a6: persistent, TMA-fed slab pipeline (default)
//   m2l_direct_kernel        a3/a4/a6: same pair arithmetic, global-memory loads (cross-check)
//   m2l_warp_kernel          a3/a4/a6 for small regions: one warp per cell, warp-level reduction of partial expansions
//   p2p_monopole_kernel      a5: monopole variant
//   dfma_peak_kernel         FP64 ALU roofline probe
//
// Staged layout of the sources (workspace), in double2 units:
//     S[z][cp][y][xpar][xh] of double2,  cp = comp >> 1 (10 pairs; slot 19 is padding),
//     xpar = x & 1, xh = x >> 1
// i.e. components are stored in pairs and each x-row is de-interleaved into its even and odd
// cells, so that the 8 lanes of a warp that share an x-parity read 8 CONSECUTIVE double2 from
// shared memory (one conflict-free 128-byte wavefront per quarter warp, LDS.128) and one 5-D
// TMA box {2, 13, 52, 10, 1} brings a whole z-slab (tile + halo) on chip.  The pair is the
// innermost tensor dimension because TMA needs the box start 16-byte aligned in the innermost
// dimension (measured: an odd FP64 start coordinate raises "illegal instruction" on sm_100a).
#pragma once

#include <cuda.h>
#include <cuda_runtime.h>
#include <stdint.h>

#include "m2l_math.cuh"
#include "taylor.cuh"

namespace octo {

constexpr int REACH_MAX = 5;            // theta_min = 0.34 for 8^3 sub-grids
constexpr int MAX_LIST = 744;           // |S_p| <= 651 for 1/3 < theta (7 * 93); + 92 near-field cells in the leaf list
constexpr int TILE_X = 16;              // target brick of one CTA pass: 16 x 8 x 3 cells = 12 warps
constexpr int TILE_Y = 8;
constexpr int TILE_Z = 3;
constexpr int NPAIR = (NCOMP + 1) / 2;  // 10 component pairs
constexpr int SLAB_XH = (TILE_X + 2 * REACH_MAX) / 2;   // 13: half-row length in the slab
constexpr int SLAB_ROW = 2 * SLAB_XH;   // 26 double2 per y-row (even half, odd half)
constexpr int SLAB_Y = TILE_Y + 2 * REACH_MAX;    // 18
constexpr int SLAB_PLANE = SLAB_Y * SLAB_ROW;     // 468 double2 per component pair
constexpr int SLAB_ELEMS = NPAIR * SLAB_PLANE;    // 4680 double2
constexpr int SLAB_BYTES = SLAB_ELEMS * 16;       // 74880 = 585 * 128 (TMA transaction size, 128-B aligned)
static_assert(SLAB_BYTES % 128 == 0, "TMA needs 128-byte aligned shared-memory destinations");
constexpr int NSTAGE = 3;
constexpr int CONSUMER_WARPS = 4 * TILE_Z;        // one warp per (xy-parity class, layer of the brick)
constexpr int STAGED_THREADS = (CONSUMER_WARPS + 1) * 32;   // + 1 producer warp
constexpr int STAGED_SMEM = NSTAGE * SLAB_BYTES + 64;
static_assert(STAGED_SMEM <= 227 * 1024, "shared memory per CTA");

struct StEntry {
    int off;                 // multipole: shared-memory offset of the source relative to the thread's base in the slab, in
                             // BYTES; monopole: offset in the mass tile (doubles, low 16 bits) + index of the weights (high 16)
    signed char dx, dy, dz, d2;   // the offset.  MULTIPOLE lists hold 8 dx, 8 dy, 8 dz: byte offsets into Params::hmul, ready
                                  // for the list walk of the slab-fed kernel (cell offsets: entry_cells());   // d2: monopole handles |Delta|^2; mixed-level lists 1 = near-field entry (not well separated);
                                  // multipole lists: the sub-grids the partners of a warp's targets fall into (bits 0-2 x, 3-5 y; MODE_TREE)
};

// Stencil tables (the interaction lists of the 8 parity classes, Eq. 15) in constant memory.  They depend on
// (theta, kind, list flavour) only and are shared by every handle of a device that uses the same lists; octo_fmm.cu
// (ConstBank) orders uploads against the kernels of other streams that still read the previous contents.  Everything
// that depends on a handle's cell width h travels in Params (kernel-parameter space), not here.
__constant__ StEntry c_entries[8 * MAX_LIST];
__constant__ int c_begin[8][2 * REACH_MAX + 2];   // first entry of (class, dz); [..][11] = end
constexpr int MAX_NEAR = 96;                      // near field (cells that are NOT well separated): <= 92 for 1/3 < theta
__constant__ char4 c_near[8][MAX_NEAR];           // (dx, dy, dz, 0) of the near-field cells of each parity class
__constant__ int c_near_count[8];

struct Params {
    int nx, ny, nz;
    int lo[3], hi[3];        // output region
    int ox, oy, oz;          // its extents
    int kb, ke;              // z-layers [kb, ke) of the output region this launch computes (staged kernel)
    int tiles_x, tiles_y, tiles_z;   // 16 x 8 x 3 bricks covering x, y of the output region and [kb, ke)
    long long ntiles;        // tiles_x * tiles_y * tiles_z
    int reach;
    const double* S;         // staged sources
    double* L;               // [20][oz][oy][ox]
    double* C;               // [3][oz][oy][ox]
    int* flags;              // flags[0] bit 0: target mass <= 0 with correction; flags[1] bit 1: some source cell has a
                             // dipole moment (raised by the staging kernel, cleared by set_moments)
    int force_dipole;        // 1: evaluate the dipole terms whatever bit 1 says
    // fused L2L epilogue of the complete solve (m2l_staged_kernel<CORR, true>): the parent level's finished expansions
    const double* pL;        // [20][nz/2][ny/2][nx/2]
    const double* pC;        // [3][...]   corrections carried beside the expansions
    const double* poff;      // [3][...]   expansion-centre offsets of the parent cells
    double hc;               // width of this level's cells
    const unsigned char* leaf;   // mixed level (m2l_staged_kernel<., ., true>): [nz][ny][nx], 1 = leaf cell
    double hmul[2 * REACH_MAX + 1];   // (double)(-d) * h for d = -5..5  (= (i_A - i_B) h), per handle
    const int* tile_list;        // levels of an adaptive tree: the bricks (ids in the dense enumeration) that have work;
                                 // nullptr = all ntiles bricks.  With a list, ntiles is its length.
    int tile_offset;             // tensor-core monopole kernels without a list: first tile of this launch (the host entry
                                 // points launch the level in chunks of z-tiles so that the copy out overlaps the rest)
    // fused L2L epilogue: extents of the parent arrays and the shift between the two index lattices,
    //   parent index = (child index >> 1) + psh   (uniform solve: pdim = n / 2, psh = 0; a level of the adaptive tree
    //   stored as a BOX of its lattice: psh = box_lo(child) / 2 - box_lo(parent))
    int pdim[3], psh[3];
    // z-slab sharding with the halo read from peer memory (f4, octo_fmm_set_neighbours): source layers exist for
    // z in [zmin, zmax]; z < 0 lies in the slab below (its layer z + nz_below), z >= nz in the slab above.  Without
    // neighbours zmin = 0, zmax = nz - 1.  nflags: the neighbours' flag words (their sources may carry dipoles).
    int zmin, zmax, nz_below;
    const int* nflags[2];
    // zr[pz] = {first, last} dz with a list entry for targets of z-parity pz (theta = 0.5: {-4, 5} for even layers, {-5, 4}
    // for odd ones): the slabs a brick streams are the union over its layers, not k0 - reach .. k0 + TILE_Z - 1 + reach
    int zr[2][2];
    // levels of an adaptive tree (with tile_list): per listed brick, which of its source layers hold anything it can meet --
    // bit i = layer k0 - REACH_MAX + i; the others are neither loaded nor walked.  nullptr = all.
    const unsigned short* tile_zmask;
};

// (double)(-d) * h for a multipole list entry's field d8 = 8 d
__device__ __forceinline__ double hmul_at(const Params& p, int d8)
{
    return *reinterpret_cast<const double*>(reinterpret_cast<const char*>(p.hmul) + 8 * REACH_MAX + d8);
}

// the z-range of source layers the brick at k0 needs (the same on the producer and the consumer side)
__device__ __forceinline__ void brick_z_range(const Params& p, int k0, int& z_lo, int& z_hi)
{
    int lo = k0 + p.zr[k0 & 1][0], hi = k0 + p.zr[k0 & 1][1];
#pragma unroll
    for (int l = 1; l < TILE_Z; ++l) {
        const int k = k0 + l;
        if (k < p.ke) { lo = min(lo, k + p.zr[k & 1][0]); hi = max(hi, k + p.zr[k & 1][1]); }
    }
    z_lo = max(lo, p.zmin);
    z_hi = min(hi, p.zmax);
}

// the tensor maps of the slab-fed kernel: the handle's own staged array and, with neighbours, theirs
struct SlabMaps { CUtensorMap own, below, above; };

// ------------------------------------------------------------------------------------------
// a2: stage the sources
// ------------------------------------------------------------------------------------------
constexpr double DIPOLE_TOL = 4.0e-16;   // |M1_i| <= DIPOLE_TOL |M| h counts as "no dipole" (round-off of a P2M / M2M about the centre of mass)

__global__ void __launch_bounds__(256) stage_multipole_kernel(const double* __restrict__ mom,
                                                              const double* __restrict__ com, double* __restrict__ S,
                                                              int nx, int ny, int nz, int z_begin, int z_count, double h,
                                                              int* __restrict__ flags, int corr)
{
    const long long ncell = (long long)nx * ny * nz;
    const long long local = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (local >= (long long)nx * ny * z_count) return;
    const long long cell = local + (long long)z_begin * ny * nx;
    const int x = (int)(cell % nx);
    const long long r = cell / nx;
    const int y = (int)(r % ny), z = (int)(r / ny);
    double M[20], s[20];
#pragma unroll
    for (int c = 0; c < 20; ++c) M[c] = mom[(long long)c * ncell + cell];
    reduce_moments(M, s, corr != 0);
    {
        const double lim = DIPOLE_TOL * fabs(M[0]) * h;
        if (fabs(M[1]) > lim || fabs(M[2]) > lim || fabs(M[3]) > lim) atomicOr(flags + 1, 2);
    }
#pragma unroll
    for (int c = 0; c < 3; ++c) s[C_DX + c] = com ? com[(long long)c * ncell + cell] : 0.0;
    s[19] = 0.0;
    const long long plane = (long long)ny * nx;   // double2 per (z, pair)
    double2* dst = reinterpret_cast<double2*>(S) + (long long)z * NPAIR * plane + (long long)y * nx + (x & 1) * (nx >> 1) + (x >> 1);
#pragma unroll
    for (int c = 0; c < NPAIR; ++c) dst[(long long)c * plane] = make_double2(s[2 * c], s[2 * c + 1]);
}

// Mixed level (f3): the leaf flag of every cell into the padding slot (component 19) of its staged record, so that the
// slab-fed kernel finds the flag of a partner next to its moments.
__global__ void __launch_bounds__(256) stage_leaf_flags_kernel(const unsigned char* __restrict__ leaf, double* __restrict__ S,
                                                               int nx, int ny, int nz)
{
    const long long cell = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (cell >= (long long)nx * ny * nz) return;
    const int x = (int)(cell % nx);
    const long long r = cell / nx;
    const int y = (int)(r % ny), z = (int)(r / ny);
    const long long plane = (long long)ny * nx;
    double2* dst = reinterpret_cast<double2*>(S) + ((long long)z * NPAIR + (NPAIR - 1)) * plane + (long long)y * nx + (x & 1) * (nx >> 1) + (x >> 1);
    dst->y = (double)leaf[cell];                // mixed level: 0 / 1 (1 = leaf); tree level: the cell's kind (0 absent, 1 leaf, 2 refined)
}

// ------------------------------------------------------------------------------------------
// PTX helpers: mbarrier + TMA
// ------------------------------------------------------------------------------------------
__device__ __forceinline__ uint32_t smem_u32(const void* p) { return (uint32_t)__cvta_generic_to_shared(p); }

__device__ __forceinline__ void mbar_init(uint64_t* bar, uint32_t count)
{
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(bar)), "r"(count) : "memory");
}
__device__ __forceinline__ void mbar_arrive_expect_tx(uint64_t* bar, uint32_t bytes)
{
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(bar)), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_arrive(uint64_t* bar)
{
    asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(smem_u32(bar)) : "memory");
}
__device__ __forceinline__ void mbar_wait(uint64_t* bar, uint32_t parity)
{
    uint32_t done;
    do {
        asm volatile(
            "{\n\t.reg .pred p;\n\t"
            "mbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n\t"
            "selp.u32 %0, 1, 0, p;\n\t}"
            : "=r"(done)
            : "r"(smem_u32(bar)), "r"(parity)
            : "memory");
    } while (!done);
}
// the producer's wait: sleeps between polls so that its spin does not take issue slots from the
// consumer warps of its sub-partition (a slab lasts ~10 us; the poll interval is ~0.25 us)
__device__ __forceinline__ void mbar_wait_backoff(uint64_t* bar, uint32_t parity)
{
    uint32_t done;
    for (;;) {
        asm volatile(
            "{\n\t.reg .pred p;\n\t"
            "mbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n\t"
            "selp.u32 %0, 1, 0, p;\n\t}"
            : "=r"(done)
            : "r"(smem_u32(bar)), "r"(parity)
            : "memory");
        if (done) break;
        __nanosleep(256);
    }
}
__device__ __forceinline__ void tma_load_slab(void* dst, const CUtensorMap* map, uint64_t* bar, int c1, int c2, int c4)
{
    asm volatile(
        "cp.async.bulk.tensor.5d.shared::cluster.global.mbarrier::complete_tx::bytes"
        " [%0], [%1, {%3, %4, %5, %6, %7}], [%2];"
        ::"r"(smem_u32(dst)), "l"((uint64_t)map), "r"(smem_u32(bar)), "r"(0), "r"(c1), "r"(c2), "r"(0), "r"(c4)
        : "memory");
}

// brick id -> lower corner; z runs fastest so that the CTAs resident at one time walk up a few
// columns and share their slabs through L2.
__device__ __forceinline__ void decode_tile(const Params& p, long long t, int& x0, int& y0, int& k0)
{
    if (p.tile_list) t = p.tile_list[t];
    k0 = p.kb + (int)(t % p.tiles_z) * TILE_Z;
    const long long c = t / p.tiles_z;
    x0 = p.lo[0] + (int)(c % p.tiles_x) * TILE_X;
    y0 = p.lo[1] + (int)(c / p.tiles_x) * TILE_Y;
}

// ------------------------------------------------------------------------------------------
// a3/a4/a6, default: persistent CTAs, one 16 x 8 x 3 target brick at a time, one cell per thread.
// Consumer warp w (< 12) holds the 32 cells of xy-parity class w & 3 in layer k0 + (w >> 2) of the
// brick (every lane of a warp runs the same interaction list, no masks); warp 12 is the TMA
// producer.  The z-slabs k0 - reach .. k0 + 2 + reach (brick + 5-cell halo in x and y, all 19
// components, 74880 bytes) are brought in by one TMA box each and are shared by the three layers:
// a warp of layer k uses slab zz with dz = zz - k when |dz| <= reach and only releases it
// otherwise.  The three slab buffers form a full/empty mbarrier ring that keeps running across
// bricks.  Twelve consumer warps (three per sub-partition) is what the FP64 pipe needs to stay
// busy at the instruction-level parallelism of the pair arithmetic (profiles/r01_*.md).
// Out-of-grid parts of a box are zero-filled by TMA = zero-mass cells with zero offset, which
// contribute exactly 0 to every coefficient (isolated boundary, L321).
// ------------------------------------------------------------------------------------------
// load the 19 staged components of one source cell (10 double2, stride `stride` double2)
#define OCTO_LOAD_SOURCE(q, stride, src, bx_, by_, bz_)                                   \
    {                                                                                     \
        double2 v_[NPAIR];                                                                \
        _Pragma("unroll") for (int c_ = 0; c_ < NPAIR; ++c_) v_[c_] = (q)[(long long)c_ * (stride)]; \
        _Pragma("unroll") for (int c_ = 0; c_ < 8; ++c_) { src[2 * c_] = v_[c_].x; src[2 * c_ + 1] = v_[c_].y; } \
        bx_ = v_[8].x; by_ = v_[8].y; bz_ = v_[9].x;                                       \
    }

// the same, plus the record's padding slot (the partner's leaf flag on a mixed level)
#define OCTO_LOAD_SOURCE_F(q, stride, src, bx_, by_, bz_, fl_)                            \
    {                                                                                     \
        double2 v_[NPAIR];                                                                \
        _Pragma("unroll") for (int c_ = 0; c_ < NPAIR; ++c_) v_[c_] = (q)[(long long)c_ * (stride)]; \
        _Pragma("unroll") for (int c_ = 0; c_ < 8; ++c_) { src[2 * c_] = v_[c_].x; src[2 * c_ + 1] = v_[c_].y; } \
        bx_ = v_[8].x; by_ = v_[8].y; bz_ = v_[9].x; fl_ = v_[9].y;                       \
    }

// the target's own expansion centre and (for the correction) M3_A / M_A in staged form
template <bool CORR>
__device__ __forceinline__ void load_target(const Params& p, int gx, int gy, int k, double (&dA)[3], double (&tA)[7])
{
    const long long plane = (long long)p.ny * p.nx;
    const double2* own = reinterpret_cast<const double2*>(p.S) + (long long)k * NPAIR * plane + (long long)gy * p.nx +
                         (gx & 1) * (p.nx >> 1) + (gx >> 1);
    const double2 d01 = own[8 * plane], d2 = own[9 * plane];
    dA[0] = d01.x; dA[1] = d01.y; dA[2] = d2.x;
    if (CORR) {
        const double mA = own[0].x;
        if (mA > 0.0) {
            const double inv = 1.0 / mA;
            const double2 o0 = own[4 * plane], o1 = own[5 * plane], o2 = own[6 * plane], o3 = own[7 * plane];
            tA[0] = o0.y * inv;                       // comp 9  (xxx)
            tA[1] = o1.x * inv; tA[2] = o1.y * inv;   // comps 10, 11
            tA[3] = o2.x * inv; tA[4] = o2.y * inv;   // comps 12, 13
            tA[5] = o3.x * inv; tA[6] = o3.y * inv;   // comps 14, 15
        } else {
            atomicOr(p.flags, 1);
        }
    }
}

// FUSE_L2L (complete solve, whole-grid output): what l2l_kernel would do in a second pass over the level is done
// here -- the correction is NOT folded into L1 but carried beside it, and the parent's expansion, Taylor-shifted to
// this cell's expansion centre, and the parent's correction are added before the one store.
template <bool CORR, bool FUSE_L2L = false>
__device__ __forceinline__ void store_target(const Params& p, const Acc& acc, const double (&tA)[7], const double (&dA)[3],
                                             int gx, int gy, int k)
{
    double L[20], C[3];
    acc_finish<CORR>(acc, tA, L, C);
    const long long ocell = (long long)p.ox * p.oy * p.oz;
    const long long o = ((long long)(k - p.lo[2]) * p.oy + (gy - p.lo[1])) * p.ox + (gx - p.lo[0]);
    if constexpr (FUSE_L2L) {
        const int pnx = p.pdim[0], pny = p.pdim[1];
        const long long pcell = (long long)pnx * pny * p.pdim[2];
        const long long P = ((long long)((k >> 1) + p.psh[2]) * pny + ((gy >> 1) + p.psh[1])) * pnx + ((gx >> 1) + p.psh[0]);
        double pL[20], sh[20], e[3];
        e[0] = ((double)(gx & 1) - 0.5) * p.hc + dA[0] - p.poff[P];
        e[1] = ((double)(gy & 1) - 0.5) * p.hc + dA[1] - p.poff[pcell + P];
        e[2] = ((double)(k & 1) - 0.5) * p.hc + dA[2] - p.poff[2 * pcell + P];
#pragma unroll
        for (int t = 0; t < 20; ++t) pL[t] = p.pL[t * pcell + P];
        taylor_shift<3>(pL, e, sh);
#pragma unroll
        for (int t = 0; t < 20; ++t) {
            double v = L[t];
            if (t >= 1 && t <= 3) v -= C[t - 1];
            L[t] = v + sh[t];
        }
#pragma unroll
        for (int c = 0; c < 3; ++c) C[c] += p.pC[c * pcell + P];
    }
#pragma unroll
    for (int c = 0; c < 20; ++c) p.L[(long long)c * ocell + o] = L[c];
#pragma unroll
    for (int c = 0; c < 3; ++c) p.C[(long long)c * ocell + o] = C[c];
}

// The consumer warps' loop over the bricks of this CTA.  DIPOLE = false is the fast path for sources
// expanded about their centre of mass (no dipole terms), see m2l_staged_kernel.
// MODE_MIXED (one level of an adaptive mesh, f3 reading R8): the lists are the leaf-level lists (Eq. 15 + near field); a
// near-field entry counts only if the target or the partner is a leaf cell -- otherwise the pair's 1/r is set to 0, and
// since every term of the pair carries a power of 1/r it contributes exactly nothing.
// MODE_TREE (a level of the adaptive tree solve, f3 reading R9): p.leaf holds the KIND of every cell (0 absent, 1 leaf,
// 2 refined); absent cells are no targets (as sources their staged record is all zeros), and two leaves do not meet here
// (they are point masses: the tensor-core leaf kernel takes them), again through 1/r = 0.  Kinds must be constant over
// sub-grids of 8^3 cells (the tree solve checks it): list entries that count for no lane of a warp are found from the
// kinds of the sub-grids around it and never fetched.
constexpr int MODE_PLAIN = 0, MODE_MIXED = 1, MODE_TREE = 2;
template <bool CORR, bool DIPOLE, bool FUSE_L2L, int MODE>
__device__ __forceinline__ void staged_consume(const Params& p, double2* slab0, uint64_t* full, uint64_t* empty, int warp, int lane)
{
    // ------------------------------ consumers ------------------------------
    const int cls_xy = warp & 3;                       // px + 2 py
    const int layer = warp >> 2;                       // 0..2
    const int px = cls_xy & 1, py = cls_xy >> 1;
    const int lx = lane & 7;
    const int ly = lane >> 3;                          // 0..3
    const int tbase = lx + 2 * ly * SLAB_ROW;          // double2

    uint32_t it = 0;
    for (long long t = blockIdx.x; t < p.ntiles; t += gridDim.x) {
        int x0, y0, k0;
        decode_tile(p, t, x0, y0, k0);
        const int k = k0 + layer;
        const int gx = x0 + px + 2 * lx, gy = y0 + py + 2 * ly;
        const bool layer_on = k < p.ke;                // warp-uniform
        const bool active = layer_on && gx < p.hi[0] && gy < p.hi[1];
        const int cls = cls_xy + ((k & 1) << 2);
        int z_lo, z_hi;
        brick_z_range(p, k0, z_lo, z_hi);
        const unsigned zmask = (MODE == MODE_TREE && p.tile_zmask) ? p.tile_zmask[t] : 0xffffu;

        double dA[3] = {0.0, 0.0, 0.0}, tA[7] = {0.0, 0.0, 0.0, 0.0, 0.0, 0.0, 0.0};
        bool leafA = false;
        bool present = active;                             // MODE_TREE: the cell exists on this level
        if (MODE == MODE_MIXED && active) leafA = p.leaf[((long long)k * p.ny + gy) * p.nx + gx] != 0;
        if (MODE == MODE_TREE && active) {
            const unsigned char kd = p.leaf[((long long)k * p.ny + gy) * p.nx + gx];
            leafA = kd == 1;
            present = kd != 0;
        }
        if (present) load_target<CORR>(p, gx, gy, k, dA, tA);
        // MODE_TREE: which list entries can count for this warp at all is known from the kinds of the SUB-GRIDS around it
        // (kinds are constant over the 8^3 cells of a sub-grid).  The warp's targets lie in two sub-grids next to each
        // other in x (lanes with lx < 4 / lx >= 4); a refined target meets every partner that exists, a leaf only refined
        // ones, an absent one nothing.  nab[sz] has bit 4 (sy + 1) + (sx + 1) set if the partners that fall into the
        // sub-grid (sx, sy, sz) away from their target's hold anything to meet; an entry knows (StEntry::d2) which (sx, sy)
        // its partners fall into, its slab which sz.  Entries that meet nothing are passed over without a load or a vote
        unsigned nab[3] = {0u, 0u, 0u};
        if constexpr (MODE == MODE_TREE) {
            const unsigned lo4 = 0x0f0f0f0fu;
            const unsigned ref = __ballot_sync(0xffffffffu, present && !leafA), lf = __ballot_sync(0xffffffffu, present && leafA);
            const int sx = (lane & 3) - 1, sy = ((lane >> 2) & 3) - 1;          // lanes 0..11: the 4 x 3 sub-grids of a layer
            const int X = ((x0 >> 3) + sx) * 8, Y = ((y0 >> 3) + sy) * 8;
#pragma unroll
            for (int c = 0; c < 3; ++c) {
                const int Z = ((k >> 3) + c - 1) * 8;
                unsigned char kd = 0;
                if (lane < 12 && layer_on && X >= 0 && Y >= 0 && Z >= 0 && X < p.nx && Y < p.ny && Z < p.nz)
                    kd = p.leaf[((long long)Z * p.ny + Y) * p.nx + X];
                const unsigned ex = __ballot_sync(0xffffffffu, kd != 0), rf = __ballot_sync(0xffffffffu, kd == 2);
                const unsigned na = (ref & lo4) ? ex : ((lf & lo4) ? rf : 0u);
                const unsigned nb = (ref & ~lo4) ? ex : ((lf & ~lo4) ? rf : 0u);
                nab[c] = (na & 0x777u) | ((nb >> 1) & 0x777u);
            }
        }
        unsigned nseg = 0u;

        Acc acc;
        acc_zero(acc);

        // Walk the slabs dz = -reach..reach of this tile and, inside each, the list segment of
        // (class, dz).  The loop is software-pipelined by hand: `fetch` loads pair s+1 from shared
        // memory and runs its head (separation, r^2, 1/r) while the body of pair s executes, so the
        // dependent head chain is hidden although only two warps share a sub-partition's FP64 pipe.
        int zz = z_lo - 1;
        int s = 0, s_end = 0;
        bool open = false;
        uint32_t b = 0;
        const double2* sl = slab0;
        double Rz0 = 0.0;
        // make (s < s_end) true by moving on to the next slab this layer uses; every slab of the
        // brick is waited for and released, used or not.  false at the end of the brick.
        auto ensure = [&]() -> bool {
          for (;;) {
            while (s >= s_end) {
                if (open) {                        // every load from this slab has been issued
                    __syncwarp();
                    if (lane == 0) mbar_arrive(&empty[b]);
                    ++it;
                    open = false;
                }
                if (++zz > z_hi) return false;
                if (MODE == MODE_TREE && !((zmask >> (zz - k0 + REACH_MAX)) & 1u)) continue;      // not loaded (producer: the same test)
                b = it % NSTAGE;
                mbar_wait(&full[b], (it / NSTAGE) & 1);
                open = true;
                const int dz = zz - k;
                if (layer_on && dz >= -p.reach && dz <= p.reach) {
                    sl = slab0 + (size_t)b * SLAB_ELEMS + tbase;
                    Rz0 = p.hmul[dz + REACH_MAX] + dA[2];
                    s = (cls * MAX_LIST + c_begin[cls][dz + REACH_MAX]) * (int)sizeof(StEntry);       // byte offsets
                    s_end = (cls * MAX_LIST + c_begin[cls][dz + REACH_MAX + 1]) * (int)sizeof(StEntry);
                    if constexpr (MODE == MODE_TREE) {
                        const int sz = ((k & 7) + dz + 8) >> 3;           // 0, 1, 2: the sub-grid layer below, of, above the target
                        nseg = sz == 0 ? nab[0] : (sz == 1 ? nab[1] : nab[2]);
                        if (nseg == 0u) s = s_end;             // nothing to meet in the sub-grid layer this slab lies in
                    }
                }
            }
            if constexpr (MODE != MODE_TREE) return true;
            else {
                // pass over the entries whose partner sub-grids hold nothing to meet (all of it warp-uniform)
                do {
                    const unsigned d2 = (unsigned)reinterpret_cast<const StEntry*>(reinterpret_cast<const char*>(c_entries) + s)->d2;
                    const unsigned pat = (d2 & 7u) * (((d2 >> 3) * 0x49u) & 0x111u);     // x bits into the rows of its y bits
                    if (pat & nseg) return true;
                    s += (int)sizeof(StEntry);
                } while (s < s_end);
            }
          }
        };
#define OCTO_FETCH(P)                                                                       \
        {                                                                                   \
            const StEntry e_ = *reinterpret_cast<const StEntry*>(reinterpret_cast<const char*>(c_entries) + s); \
            s += (int)sizeof(StEntry);                                                      \
            const double2* q_ = reinterpret_cast<const double2*>(reinterpret_cast<const char*>(sl) + e_.off); \
            double bx_, by_, bz_, fl_ = 0.0;                                                \
            if (MODE != MODE_PLAIN) { OCTO_LOAD_SOURCE_F(q_, SLAB_PLANE, P.src, bx_, by_, bz_, fl_); } \
            else       { OCTO_LOAD_SOURCE(q_, SLAB_PLANE, P.src, bx_, by_, bz_); }          \
            P.x = hmul_at(p, e_.dx) + (dA[0] - bx_);                                        \
            P.y = hmul_at(p, e_.dy) + (dA[1] - by_);                                        \
            P.z = Rz0 - bz_;                                                                \
            P.w = pair_head(P.x, P.y, P.z);                                                 \
            if (MODE == MODE_MIXED && e_.d2 && !leafA && fl_ == 0.0) P.w = 0.0;             \
            /* MODE_TREE: the partner is absent, or a leaf meets a leaf -> this lane takes nothing */ \
            if (MODE == MODE_TREE && (!present || fl_ == 0.0 || (leafA && fl_ == 1.0))) P.w = 0.0; \
        }
        struct Fetched { double src[16]; double x, y, z, w; } A, B;
#define OCTO_BODY(P) m2l_pair<CORR, DIPOLE>(acc, P.x, P.y, P.z, P.w, P.src, tA)
        // the loop over the entries, software-pipelined two deep (see above); a lane whose pair does not count has 1/r = 0
#define OCTO_LOOP()                                                                         \
        if (ensure()) {                                                                     \
            OCTO_FETCH(A);                                                                  \
            for (;;) {                                                                      \
                if (!ensure()) break;                                                       \
                OCTO_FETCH(B);                                                              \
                OCTO_BODY(A);                                                               \
                if (!ensure()) { A = B; break; }                                            \
                OCTO_FETCH(A);                                                              \
                OCTO_BODY(B);                                                               \
            }                                                                               \
            OCTO_BODY(A);                                                                   \
        }
        bool leaf_warp = false;
        if constexpr (MODE == MODE_TREE) leaf_warp = __all_sync(0xffffffffu, !present || leafA);
        if (leaf_warp) {
            // MODE_TREE, a warp of LEAF targets (the shell of leaves around a refined region: most bricks of a level).  A
            // leaf has no children: of its expansion only L0 and L1 (+ correction) are ever used -- the leaf finish evaluates
            // them at the cell centre.  The order-2 and order-3 sums are discarded after the loop, which makes them dead:
            // the compiler drops their instructions from this copy of the loop (83 instead of 117 per pair)
            OCTO_LOOP()
#pragma unroll
            for (int i = 0; i < 5; ++i) acc.l2[i] = 0.0;
#pragma unroll
            for (int i = 0; i < 7; ++i) acc.l3[i] = 0.0;
        } else {
            OCTO_LOOP()
        }
#undef OCTO_LOOP
#undef OCTO_BODY
#undef OCTO_FETCH

        if (present) store_target<CORR, FUSE_L2L>(p, acc, tA, dA, gx, gy, k);
    }
}

template <bool CORR, bool FUSE_L2L = false, int MODE = MODE_PLAIN>
__global__ void __launch_bounds__(STAGED_THREADS, 1)
m2l_staged_kernel(const __grid_constant__ SlabMaps maps, const __grid_constant__ Params p)
{
    extern __shared__ __align__(128) unsigned char smem_raw[];
    double2* slab0 = reinterpret_cast<double2*>(smem_raw);
    uint64_t* full = reinterpret_cast<uint64_t*>(smem_raw + NSTAGE * SLAB_BYTES);
    uint64_t* empty = full + NSTAGE;

    const int warp = __shfl_sync(0xffffffffu, (int)(threadIdx.x >> 5), 0);
    const int lane = threadIdx.x & 31;

    if (threadIdx.x == 0) {
        for (int b = 0; b < NSTAGE; ++b) {
            mbar_init(&full[b], 1);
            mbar_init(&empty[b], CONSUMER_WARPS);
        }
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
        asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
    }
    __syncthreads();

    if (warp == CONSUMER_WARPS) {
        // ------------------------------ producer ------------------------------
        if (lane == 0) {
            uint32_t it = 0;
            for (long long t = blockIdx.x; t < p.ntiles; t += gridDim.x) {
                int x0, y0, k0;
                decode_tile(p, t, x0, y0, k0);
                int z_lo, z_hi;
                brick_z_range(p, k0, z_lo, z_hi);
                const unsigned zmask = (MODE == MODE_TREE && p.tile_zmask) ? p.tile_zmask[t] : 0xffffu;
                for (int zz = z_lo; zz <= z_hi; ++zz) {
                    if (MODE == MODE_TREE && !((zmask >> (zz - k0 + REACH_MAX)) & 1u)) continue;
                    const uint32_t b = it % NSTAGE;
                    if (it >= NSTAGE) mbar_wait_backoff(&empty[b], ((it / NSTAGE) - 1) & 1);
                    mbar_arrive_expect_tx(&full[b], SLAB_BYTES);
                    // a layer of a neighbouring z-slab comes straight from that rank's staged array (peer memory)
                    const CUtensorMap* m = &maps.own;
                    int zc = zz;
                    if (zz < 0) { m = &maps.below; zc = zz + p.nz_below; }
                    else if (zz >= p.nz) { m = &maps.above; zc = zz - p.nz; }
                    tma_load_slab(slab0 + (size_t)b * SLAB_ELEMS, m, &full[b], (x0 >> 1) - 3, 2 * (y0 - REACH_MAX), zc);
                    ++it;
                }
            }
        }
        return;
    }

    // ------------------------------ consumers ------------------------------
    // Sources expanded about their centre of mass have no dipole moment: the staging kernel raises bit 1 of
    // the flags if any cell has |M1_i| > DIPOLE_TOL |M| h, and only then (or when the caller forces it) the
    // 27 dipole terms are evaluated.  The branch is uniform over the grid.
    bool dipole = p.force_dipole || ((*(volatile const int*)(p.flags + 1)) & 2);
    if (p.nflags[0] && ((*(volatile const int*)(p.nflags[0] + 1)) & 2)) dipole = true;
    if (p.nflags[1] && ((*(volatile const int*)(p.nflags[1] + 1)) & 2)) dipole = true;
    if (dipole) staged_consume<CORR, true, FUSE_L2L, MODE>(p, slab0, full, empty, warp, lane);
    else        staged_consume<CORR, false, FUSE_L2L, MODE>(p, slab0, full, empty, warp, lane);
}

// ------------------------------------------------------------------------------------------
// a3/a4/a6, cross-check variant: one thread per target cell, sources read straight from the
// staged array in global memory with explicit in-grid tests.  Same pair arithmetic.
// Block = 256 threads = the 8 parity classes x 32 cells of a 16 x 8 x 2 brick, two passes in z.
// ------------------------------------------------------------------------------------------
template <bool CORR>
__global__ void __launch_bounds__(256) m2l_direct_kernel(const __grid_constant__ Params p)
{
    const int warp = __shfl_sync(0xffffffffu, (int)(threadIdx.x >> 5), 0);
    const int lane = threadIdx.x & 31;
    const int px = warp & 1, py = (warp >> 1) & 1, pz = warp >> 2;
    const int bx = (p.ox + 15) / 16, by = (p.oy + 7) / 8;
    const int b = blockIdx.x;
    const int x0 = p.lo[0] + (b % bx) * 16, y0 = p.lo[1] + ((b / bx) % by) * 8, z0 = p.lo[2] + (b / (bx * by)) * 4;
    const int gx = x0 + px + 2 * (lane & 7), gy = y0 + py + 2 * (lane >> 3);
    const long long plane = (long long)p.ny * p.nx;
    const double2* S2 = reinterpret_cast<const double2*>(p.S);
    const int cls = warp;
    const bool dipole = p.force_dipole || ((*(volatile const int*)(p.flags + 1)) & 2);
    for (int pass = 0; pass < 2; ++pass) {
        const int k = z0 + pz + 2 * pass;
        if (!(gx < p.hi[0] && gy < p.hi[1] && k < p.hi[2])) continue;
        double dA[3] = {0.0, 0.0, 0.0}, tA[7] = {0.0, 0.0, 0.0, 0.0, 0.0, 0.0, 0.0};
        load_target<CORR>(p, gx, gy, k, dA, tA);
        Acc acc;
        acc_zero(acc);
        const int s_end = c_begin[cls][2 * REACH_MAX + 1];
#pragma unroll 1
        for (int s = c_begin[cls][0]; s < s_end; ++s) {
            const StEntry e = c_entries[cls * MAX_LIST + s];
            const int sx = gx + (e.dx >> 3), sy = gy + (e.dy >> 3), sz = k + (e.dz >> 3);
            if (sx < 0 || sy < 0 || sz < 0 || sx >= p.nx || sy >= p.ny || sz >= p.nz) continue;
            const double2* q = S2 + (long long)sz * NPAIR * plane + (long long)sy * p.nx + (sx & 1) * (p.nx >> 1) + (sx >> 1);
            double src[16], bx_, by_, bz_;
            OCTO_LOAD_SOURCE(q, plane, src, bx_, by_, bz_);
            const double x = hmul_at(p, e.dx) + (dA[0] - bx_);
            const double y = hmul_at(p, e.dy) + (dA[1] - by_);
            const double z = hmul_at(p, e.dz) + (dA[2] - bz_);
            if (dipole) m2l_pair<CORR, true>(acc, x, y, z, pair_head(x, y, z), src, tA);
            else        m2l_pair<CORR, false>(acc, x, y, z, pair_head(x, y, z), src, tA);
        }
        store_target<CORR>(p, acc, tA, dA, gx, gy, k);
    }
}

// ------------------------------------------------------------------------------------------
// One level of an adaptive mesh (reading R8): the near-field pairs.  leaf[cell] = 1: the cell
// belongs to a leaf sub-grid (no children).  A pair that is not well separated is normally left to the children; when A or
// B has none it is taken at this level with the same pair formula.  Runs AFTER an interaction kernel has written the
// Eq. 15 part: one thread per target cell (warps = parity classes as in m2l_direct_kernel), the near-field cells B with
// leaf[A] | leaf[B] are accumulated and the finished coefficients are ADDED to L and Lcorr (acc_finish is linear).
// count (may be null): number of pairs taken, for the bit-exact check of the pair set.
// ------------------------------------------------------------------------------------------
template <bool CORR>
__global__ void __launch_bounds__(256) m2l_near_kernel(const __grid_constant__ Params p, const unsigned char* __restrict__ leaf,
                                                       unsigned long long* __restrict__ count)
{
    const int warp = __shfl_sync(0xffffffffu, (int)(threadIdx.x >> 5), 0);
    const int lane = threadIdx.x & 31;
    const int px = warp & 1, py = (warp >> 1) & 1, pz = warp >> 2;
    const int bx = (p.ox + 15) / 16, by = (p.oy + 7) / 8;
    const int b = blockIdx.x;
    const int x0 = p.lo[0] + (b % bx) * 16, y0 = p.lo[1] + ((b / bx) % by) * 8, z0 = p.lo[2] + (b / (bx * by)) * 4;
    const int gx = x0 + px + 2 * (lane & 7), gy = y0 + py + 2 * (lane >> 3);
    const long long plane = (long long)p.ny * p.nx;
    const double2* S2 = reinterpret_cast<const double2*>(p.S);
    const int cls = warp;
    const long long ocell = (long long)p.ox * p.oy * p.oz;
    const bool dipole = p.force_dipole || ((*(volatile const int*)(p.flags + 1)) & 2);   // as the interaction kernels
    unsigned long long taken = 0;
    for (int pass = 0; pass < 2; ++pass) {
        const int k = z0 + pz + 2 * pass;
        if (!(gx < p.hi[0] && gy < p.hi[1] && k < p.hi[2])) continue;
        const bool leafA = leaf[(long long)k * plane + (long long)gy * p.nx + gx] != 0;
        double dA[3] = {0.0, 0.0, 0.0}, tA[7] = {0.0, 0.0, 0.0, 0.0, 0.0, 0.0, 0.0};
        load_target<CORR>(p, gx, gy, k, dA, tA);
        Acc acc;
        acc_zero(acc);
        const int n_near = c_near_count[cls];
        bool any = false;
#pragma unroll 1
        for (int s = 0; s < n_near; ++s) {
            const char4 e = c_near[cls][s];
            const int sx = gx + e.x, sy = gy + e.y, sz = k + e.z;
            if (sx < 0 || sy < 0 || sz < 0 || sx >= p.nx || sy >= p.ny || sz >= p.nz) continue;
            if (!leafA && leaf[(long long)sz * plane + (long long)sy * p.nx + sx] == 0) continue;
            const double2* q = S2 + (long long)sz * NPAIR * plane + (long long)sy * p.nx + (sx & 1) * (p.nx >> 1) + (sx >> 1);
            double src[16], bx_, by_, bz_;
            OCTO_LOAD_SOURCE(q, plane, src, bx_, by_, bz_);
            const double x = p.hmul[e.x + REACH_MAX] + (dA[0] - bx_);
            const double y = p.hmul[e.y + REACH_MAX] + (dA[1] - by_);
            const double z = p.hmul[e.z + REACH_MAX] + (dA[2] - bz_);
            if (dipole) m2l_pair<CORR, true>(acc, x, y, z, pair_head(x, y, z), src, tA);
            else        m2l_pair<CORR, false>(acc, x, y, z, pair_head(x, y, z), src, tA);
            any = true;
            ++taken;
        }
        if (any) {
            double L[20], C[3];
            acc_finish<CORR>(acc, tA, L, C);
            const long long o = ((long long)(k - p.lo[2]) * p.oy + (gy - p.lo[1])) * p.ox + (gx - p.lo[0]);
#pragma unroll
            for (int c = 0; c < 20; ++c) p.L[(long long)c * ocell + o] += L[c];
#pragma unroll
            for (int c = 0; c < 3; ++c) p.C[(long long)c * ocell + o] += C[c];
        }
    }
    if (count) {
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) taken += __shfl_xor_sync(0xffffffffu, taken, o);
        if (lane == 0 && taken) atomicAdd(count, taken);
    }
}

// ------------------------------------------------------------------------------------------
// a3/a4/a6 for small output regions (coarse levels of the complete solve, single sub-grids):
// one WARP per target cell.  The lanes split the cell's interaction list (entry s = lane, lane + 32,
// ...), each accumulates a partial expansion, and the 20 + 3 partial sums are combined by a
// butterfly of warp shuffles; lane 0 stores.  With a few hundred to a few thousand targets the
// one-cell-per-thread kernels leave most SMs idle and take ~150 us of pure latency; this takes
// ~10 us.  Sources are read from the staged array in global memory with explicit in-grid tests.
// ------------------------------------------------------------------------------------------
template <bool CORR>
__global__ void __launch_bounds__(256) m2l_warp_kernel(const __grid_constant__ Params p)
{
    const int warp = __shfl_sync(0xffffffffu, (int)(threadIdx.x >> 5), 0);
    const int lane = threadIdx.x & 31;
    const long long t = (long long)blockIdx.x * 8 + warp;
    if (t >= (long long)p.ox * p.oy * p.oz) return;
    const int gx = p.lo[0] + (int)(t % p.ox), gy = p.lo[1] + (int)((t / p.ox) % p.oy), k = p.lo[2] + (int)(t / ((long long)p.ox * p.oy));
    const int cls = (gx & 1) + 2 * (gy & 1) + 4 * (k & 1);
    const long long plane = (long long)p.ny * p.nx;
    const double2* S2 = reinterpret_cast<const double2*>(p.S);
    const bool dipole = p.force_dipole || ((*(volatile const int*)(p.flags + 1)) & 2);
    double dA[3] = {0.0, 0.0, 0.0}, tA[7] = {0.0, 0.0, 0.0, 0.0, 0.0, 0.0, 0.0};
    load_target<CORR>(p, gx, gy, k, dA, tA);
    Acc acc;
    acc_zero(acc);
    const int s_end = c_begin[cls][2 * REACH_MAX + 1];
#pragma unroll 1
    for (int s = c_begin[cls][0] + lane; s < s_end; s += 32) {
        const StEntry e = c_entries[cls * MAX_LIST + s];
        const int sx = gx + (e.dx >> 3), sy = gy + (e.dy >> 3), sz = k + (e.dz >> 3);
        if (sx < 0 || sy < 0 || sz < 0 || sx >= p.nx || sy >= p.ny || sz >= p.nz) continue;
        const double2* q = S2 + (long long)sz * NPAIR * plane + (long long)sy * p.nx + (sx & 1) * (p.nx >> 1) + (sx >> 1);
        double src[16], bx_, by_, bz_;
        OCTO_LOAD_SOURCE(q, plane, src, bx_, by_, bz_);
        const double x = hmul_at(p, e.dx) + (dA[0] - bx_);
        const double y = hmul_at(p, e.dy) + (dA[1] - by_);
        const double z = hmul_at(p, e.dz) + (dA[2] - bz_);
        if (dipole) m2l_pair<CORR, true>(acc, x, y, z, pair_head(x, y, z), src, tA);
        else        m2l_pair<CORR, false>(acc, x, y, z, pair_head(x, y, z), src, tA);
    }
    // warp-level reduction of the partial expansions (fixed butterfly order: deterministic)
    double* v = reinterpret_cast<double*>(&acc);
#pragma unroll
    for (int c = 0; c < ACC_DOUBLES; ++c) {
        double a = v[c];
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) a += __shfl_xor_sync(0xffffffffu, a, o);
        v[c] = a;
    }
    if (lane == 0) store_target<CORR>(p, acc, tA, dA, gx, gy, k);
}

// ------------------------------------------------------------------------------------------
// Two right-hand sides in ONE pass (Alg. 1: "Compute g, phi, and d(phi)/dt using
// the FMM"): the density (sources p.S, correction as configured) and its time derivative (sources S2: the moments of
// d(rho)/dt about the SAME centres, staged with the correction off; no correction, dipole terms always) share the
// interaction list, the separation R, 1/|R| and the radial factors of every pair; each keeps its own accumulators and
// its own pair body.  Outputs: p.L / p.C for the density, q.L / q.C for the second right-hand side (q.C gets zeros).
// m2l_warp2_kernel: one warp per target cell (coarse levels); m2l_direct2_kernel: one thread per target cell, sources
// from global memory (the measured variant for the fine levels).
// ------------------------------------------------------------------------------------------
#define OCTO_LOAD_SOURCE2(q, stride, src)                                                  \
    {                                                                                     \
        double2 v_[8];                                                                    \
        _Pragma("unroll") for (int c_ = 0; c_ < 8; ++c_) v_[c_] = (q)[(long long)c_ * (stride)]; \
        _Pragma("unroll") for (int c_ = 0; c_ < 8; ++c_) { src[2 * c_] = v_[c_].x; src[2 * c_ + 1] = v_[c_].y; } \
    }

template <bool CORR>
__global__ void __launch_bounds__(256) m2l_warp2_kernel(const __grid_constant__ Params p, const __grid_constant__ Params q)
{
    const int warp = __shfl_sync(0xffffffffu, (int)(threadIdx.x >> 5), 0);
    const int lane = threadIdx.x & 31;
    const long long t = (long long)blockIdx.x * 8 + warp;
    if (t >= (long long)p.ox * p.oy * p.oz) return;
    const int gx = p.lo[0] + (int)(t % p.ox), gy = p.lo[1] + (int)((t / p.ox) % p.oy), k = p.lo[2] + (int)(t / ((long long)p.ox * p.oy));
    const int cls = (gx & 1) + 2 * (gy & 1) + 4 * (k & 1);
    const long long plane = (long long)p.ny * p.nx;
    const double2* S1 = reinterpret_cast<const double2*>(p.S);
    const double2* S2 = reinterpret_cast<const double2*>(q.S);
    const bool dipole = p.force_dipole || ((*(volatile const int*)(p.flags + 1)) & 2);
    double dA[3] = {0.0, 0.0, 0.0}, tA[7] = {0.0, 0.0, 0.0, 0.0, 0.0, 0.0, 0.0};
    const double t0[7] = {0.0, 0.0, 0.0, 0.0, 0.0, 0.0, 0.0};
    load_target<CORR>(p, gx, gy, k, dA, tA);
    Acc acc, acc2;
    acc_zero(acc);
    acc_zero(acc2);
    const int s_end = c_begin[cls][2 * REACH_MAX + 1];
#pragma unroll 1
    for (int s = c_begin[cls][0] + lane; s < s_end; s += 32) {
        const StEntry e = c_entries[cls * MAX_LIST + s];
        const int sx = gx + (e.dx >> 3), sy = gy + (e.dy >> 3), sz = k + (e.dz >> 3);
        if (sx < 0 || sy < 0 || sz < 0 || sx >= p.nx || sy >= p.ny || sz >= p.nz) continue;
        const long long o = (long long)sz * NPAIR * plane + (long long)sy * p.nx + (sx & 1) * (p.nx >> 1) + (sx >> 1);
        double src[16], src2[16], bx_, by_, bz_;
        OCTO_LOAD_SOURCE(S1 + o, plane, src, bx_, by_, bz_);
        OCTO_LOAD_SOURCE2(S2 + o, plane, src2);
        const double x = hmul_at(p, e.dx) + (dA[0] - bx_);
        const double y = hmul_at(p, e.dy) + (dA[1] - by_);
        const double z = hmul_at(p, e.dz) + (dA[2] - bz_);
        const double w = pair_head(x, y, z);
        if (dipole) m2l_pair<CORR, true>(acc, x, y, z, w, src, tA);
        else        m2l_pair<CORR, false>(acc, x, y, z, w, src, tA);
        m2l_pair<false, true>(acc2, x, y, z, w, src2, t0);
    }
    double* v = reinterpret_cast<double*>(&acc);
    double* v2 = reinterpret_cast<double*>(&acc2);
#pragma unroll
    for (int c = 0; c < ACC_DOUBLES; ++c) {
        double a = v[c], b = v2[c];
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) {
            a += __shfl_xor_sync(0xffffffffu, a, o);
            b += __shfl_xor_sync(0xffffffffu, b, o);
        }
        v[c] = a;
        v2[c] = b;
    }
    if (lane == 0) {
        store_target<CORR>(p, acc, tA, dA, gx, gy, k);
        store_target<false>(q, acc2, t0, dA, gx, gy, k);
    }
}

template <bool CORR>
__global__ void __launch_bounds__(256) m2l_direct2_kernel(const __grid_constant__ Params p, const __grid_constant__ Params q)
{
    const int warp = __shfl_sync(0xffffffffu, (int)(threadIdx.x >> 5), 0);
    const int lane = threadIdx.x & 31;
    const int px = warp & 1, py = (warp >> 1) & 1, pz = warp >> 2;
    const int bx = (p.ox + 15) / 16, by = (p.oy + 7) / 8;
    const int b = blockIdx.x;
    const int x0 = p.lo[0] + (b % bx) * 16, y0 = p.lo[1] + ((b / bx) % by) * 8, z0 = p.lo[2] + (b / (bx * by)) * 4;
    const int gx = x0 + px + 2 * (lane & 7), gy = y0 + py + 2 * (lane >> 3);
    const long long plane = (long long)p.ny * p.nx;
    const double2* S1 = reinterpret_cast<const double2*>(p.S);
    const double2* S2 = reinterpret_cast<const double2*>(q.S);
    const int cls = warp;
    const bool dipole = p.force_dipole || ((*(volatile const int*)(p.flags + 1)) & 2);
    const double t0[7] = {0.0, 0.0, 0.0, 0.0, 0.0, 0.0, 0.0};
    for (int pass = 0; pass < 2; ++pass) {
        const int k = z0 + pz + 2 * pass;
        if (!(gx < p.hi[0] && gy < p.hi[1] && k < p.hi[2])) continue;
        double dA[3] = {0.0, 0.0, 0.0}, tA[7] = {0.0, 0.0, 0.0, 0.0, 0.0, 0.0, 0.0};
        load_target<CORR>(p, gx, gy, k, dA, tA);
        Acc acc, acc2;
        acc_zero(acc);
        acc_zero(acc2);
        const int s_end = c_begin[cls][2 * REACH_MAX + 1];
#pragma unroll 1
        for (int s = c_begin[cls][0]; s < s_end; ++s) {
            const StEntry e = c_entries[cls * MAX_LIST + s];
            const int sx = gx + (e.dx >> 3), sy = gy + (e.dy >> 3), sz = k + (e.dz >> 3);
            if (sx < 0 || sy < 0 || sz < 0 || sx >= p.nx || sy >= p.ny || sz >= p.nz) continue;
            const long long o = (long long)sz * NPAIR * plane + (long long)sy * p.nx + (sx & 1) * (p.nx >> 1) + (sx >> 1);
            double src[16], src2[16], bx_, by_, bz_;
            OCTO_LOAD_SOURCE(S1 + o, plane, src, bx_, by_, bz_);
            OCTO_LOAD_SOURCE2(S2 + o, plane, src2);
            const double x = hmul_at(p, e.dx) + (dA[0] - bx_);
            const double y = hmul_at(p, e.dy) + (dA[1] - by_);
            const double z = hmul_at(p, e.dz) + (dA[2] - bz_);
            const double w = pair_head(x, y, z);
            if (dipole) m2l_pair<CORR, true>(acc, x, y, z, w, src, tA);
            else        m2l_pair<CORR, false>(acc, x, y, z, w, src, tA);
            m2l_pair<false, true>(acc2, x, y, z, w, src2, t0);
        }
        store_target<CORR>(p, acc, tA, dA, gx, gy, k);
        store_target<false>(q, acc2, t0, dA, gx, gy, k);
    }
}

// ------------------------------------------------------------------------------------------
// a5: monopole (leaf) variant.  R = (i_A - i_B) h has no per-cell part, so -1/|R| and
// -R/|R|^3 depend on the offset Delta only: they are tabulated for the 11^3 offsets on the host
// in FP64 and the kernel is a 4-FMA stencil sum.
// The mass is staged zero-padded by REACH_MAX cells (x: 5 on the left, 7 on the right, so that a half-row is a
// multiple of 16 bytes) and with every x-row de-interleaved into its even and odd cells:
//   P[z + 5][y + 5][xpar][xh],  padded x = x + 5, xpar = padded x & 1, xh = padded x >> 1,  MONO_PADX = nx + 12
// -- the layout the interaction kernel wants in shared memory, so that one TMA box brings a whole tile.
// ------------------------------------------------------------------------------------------
constexpr int MONO_PAD_RIGHT = REACH_MAX + 2;
__global__ void __launch_bounds__(256) stage_monopole_kernel(const double* __restrict__ mass, double* __restrict__ P,
                                                             int nx, int ny, int nz)
{
    const int X = nx + REACH_MAX + MONO_PAD_RIGHT, Y = ny + 2 * REACH_MAX, Z = nz + 2 * REACH_MAX;
    const long long n = (long long)X * Y * Z;
    const long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x;     // padded cell index, x fastest
    if (i >= n) return;
    const int xp = (int)(i % X);
    const long long r = i / X;
    const int x = xp - REACH_MAX, y = (int)(r % Y) - REACH_MAX, z = (int)(r / Y) - REACH_MAX;
    const bool in = x >= 0 && y >= 0 && z >= 0 && x < nx && y < ny && z < nz;
    P[r * X + (xp & 1) * (X >> 1) + (xp >> 1)] = in ? mass[((long long)z * ny + y) * nx + x] : 0.0;
}

constexpr int MT_X = 16, MT_Y = 16, MT_Z = 16;          // target tile of one block
constexpr int MS_X = MT_X + 2 * REACH_MAX, MS_Y = MT_Y + 2 * REACH_MAX, MS_Z = MT_Z + 2 * REACH_MAX;
constexpr int MS_XH = 14;                               // half-row: 13 cells of one x-parity + 1 pad
constexpr int MS_ROW = 2 * MS_XH;                       // 28 doubles: two tile rows are 64 bytes mod 128 apart
constexpr int MONO_TILE_BYTES = MS_ROW * MS_Y * MS_Z * 8;                    // 151424 B
constexpr int MONO_NW = (2 * REACH_MAX + 1) * (2 * REACH_MAX + 1) * (2 * REACH_MAX + 1);   // 1331 offsets Delta
constexpr int MONO_SMEM = MONO_TILE_BYTES + MONO_NW * 32 + 64;               // + 42592 B of weights + mbarrier = 194080 B
constexpr int MONO_THREADS = 512;
static_assert(MONO_SMEM <= 227 * 1024, "shared memory per CTA");

// One block (16 warps, one per SM) = a 16 x 16 x 16 target tile.  Shared memory holds the masses of the tile + 5-cell
// halo (every x-row de-interleaved into its even and odd cells and padded to 28 doubles: the 32 lanes of a warp --
// 8 cells two apart in x, 4 rows two apart in y -- read 256 consecutive-bank bytes, two conflict-free wavefronts per
// LDS.64) and the table of the weights (-1/|R|, -R/|R|^3) of all 11^3 offsets Delta (R = -Delta h has no per-cell
// part; built on the host in FP64).  Warp w: xy-parity class (w >> 1) & 3, rows 4 (w & 1) + {0..3} of that class,
// layers 8 (w >> 3) + {0..7}; a thread owns one (x, y) and 8 layers: two passes (even z, odd z) of 4 targets that
// share the parity class, hence the list entry, its tile offset and its weights.  Per entry and warp: one constant
// load (tile offset and weight index, packed on the host), two broadcast LDS.128 of the weights, four LDS.64 of the
// masses, 16 DFMAs.
__device__ __forceinline__ void tma_load_tile3(void* dst, const CUtensorMap* map, uint64_t* bar, int c0, int c1, int c2)
{
    asm volatile(
        "cp.async.bulk.tensor.3d.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1, {%3, %4, %5}], [%2];"
        ::"r"(smem_u32(dst)), "l"((uint64_t)map), "r"(smem_u32(bar)), "r"(c0), "r"(c1), "r"(c2)
        : "memory");
}

__global__ void __launch_bounds__(MONO_THREADS, 1) p2p_monopole_kernel(const __grid_constant__ CUtensorMap tmap, const Params p,
                                                                       const double4* __restrict__ Wg, double* __restrict__ out)
{
    extern __shared__ __align__(128) unsigned char mono_smem[];
    double* tile = reinterpret_cast<double*>(mono_smem);
    double4* W = reinterpret_cast<double4*>(mono_smem + MONO_TILE_BYTES);
    const int warp = __shfl_sync(0xffffffffu, (int)(threadIdx.x >> 5), 0);
    const int lane = threadIdx.x & 31;
    const int px = (warp >> 1) & 1, py = (warp >> 2) & 1, zg = warp >> 3;
    const int bx = (p.ox + MT_X - 1) / MT_X, by = (p.oy + MT_Y - 1) / MT_Y;
    const int b = blockIdx.x;
    const int x0 = p.lo[0] + (b % bx) * MT_X, y0 = p.lo[1] + ((b / bx) % by) * MT_Y, z0 = p.lo[2] + (b / (bx * by)) * MT_Z;
    uint64_t* bar = reinterpret_cast<uint64_t*>(mono_smem + MONO_TILE_BYTES + MONO_NW * 32);

    // the tile (x0-5 .. x0+22, y0-5 .. y0+20, z0-5 .. z0+20 = staged coordinates x0.., y0.., z0..) is ONE TMA box
    // {14, 52, 26} of the staged array [z][y * 2 + xpar][xh]; parts beyond the array are zero-filled
    if (threadIdx.x == 0) {
        mbar_init(bar, 1);
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
        asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
        mbar_arrive_expect_tx(bar, MONO_TILE_BYTES);
        tma_load_tile3(tile, &tmap, bar, x0 >> 1, 2 * y0, z0);
    }
    for (int i = threadIdx.x; i < MONO_NW; i += MONO_THREADS) W[i] = Wg[i];
    __syncthreads();                 // weights in place, barrier initialised
    mbar_wait(bar, 0);               // tile in place

    const int lx = lane & 7, ly = ((warp & 1) << 2) + (lane >> 3);
    const int gx = x0 + px + 2 * lx, gy = y0 + py + 2 * ly;
    const bool act_xy = gx < p.hi[0] && gy < p.hi[1];
    const long long ocell = (long long)p.ox * p.oy * p.oz;
    constexpr int LAYER2 = 2 * MS_Y * MS_ROW;
#pragma unroll 1
    for (int pz = 0; pz < 2; ++pz) {
        const int cls = (px + 2 * py) + 4 * pz;
        // the entry offsets carry the x-parity part (host: e.off), the thread adds its own layer, row and half-row index
        const double* base = tile + ((8 * zg + pz + REACH_MAX) * MS_Y + (py + 2 * ly + REACH_MAX)) * MS_ROW + lx;
        double a[4][4];
#pragma unroll
        for (int j = 0; j < 4; ++j)
#pragma unroll
            for (int c = 0; c < 4; ++c) a[j][c] = 0.0;
        const int s_begin = cls * MAX_LIST + c_begin[cls][0], s_end = cls * MAX_LIST + c_begin[cls][2 * REACH_MAX + 1];
#pragma unroll 2
        for (int s = s_begin; s < s_end; ++s) {
            const int packed = c_entries[s].off;                 // low 16 bits: tile offset (signed), high 16: weight index
            const double* q = base + (short)(packed & 0xffff);
            const double4 w = W[packed >> 16];
            const double m0 = q[0], m1 = q[LAYER2], m2 = q[2 * LAYER2], m3 = q[3 * LAYER2];
            // boustrophedon order: consecutive DFMAs share the mass or the weight, so that one operand always
            // comes from the operand-reuse cache (a DFMA with three fresh register operands takes 3 cycles, not 2)
            a[0][0] = fma(m0, w.x, a[0][0]); a[0][1] = fma(m0, w.y, a[0][1]); a[0][2] = fma(m0, w.z, a[0][2]); a[0][3] = fma(m0, w.w, a[0][3]);
            a[1][3] = fma(m1, w.w, a[1][3]); a[1][2] = fma(m1, w.z, a[1][2]); a[1][1] = fma(m1, w.y, a[1][1]); a[1][0] = fma(m1, w.x, a[1][0]);
            a[2][0] = fma(m2, w.x, a[2][0]); a[2][1] = fma(m2, w.y, a[2][1]); a[2][2] = fma(m2, w.z, a[2][2]); a[2][3] = fma(m2, w.w, a[2][3]);
            a[3][3] = fma(m3, w.w, a[3][3]); a[3][2] = fma(m3, w.z, a[3][2]); a[3][1] = fma(m3, w.y, a[3][1]); a[3][0] = fma(m3, w.x, a[3][0]);
        }
#pragma unroll
        for (int j = 0; j < 4; ++j) {
            const int k = z0 + 8 * zg + pz + 2 * j;
            if (act_xy && k < p.hi[2]) {
                const long long o = ((long long)(k - p.lo[2]) * p.oy + (gy - p.lo[1])) * p.ox + (gx - p.lo[0]);
#pragma unroll
                for (int c = 0; c < 4; ++c) out[c * ocell + o] = a[j][c];
            }
        }
    }
}

// ------------------------------------------------------------------------------------------
// a5 on the FP64 tensor-core instruction (DMMA m8n8k4), the default monopole kernel.
//
// The monopole sum is a convolution, out[c][t] = sum_s W[c][s] m[t + s] with weights that depend on the offset only,
// i.e. a dense contraction, and `mma.sync.m8n8k4.f64` runs on the FP64 pipe at 8 FMAs per lane for FOUR register
// operands -- measured 37.2 TFLOP/s on this B200 (100 % of the FP64 peak), where a DFMA with three fresh register
// operands reaches 65 % (register-file read bandwidth).  One DMMA, D(8x8) += A(8x4) B(4x8):
//   columns j : 8 targets two apart in x (the x-even cells of a 16-cell row segment)
//   k         : 4 source offsets s_k;  B[k][j] = m[t_j + s_k]
//   rows i    : component c = i & 3 of (phi, gx, gy, gz) for variant v = i >> 2; v = 0 is the target t_j itself,
//               v = 1 its x-odd sibling t_j + e_x, for which the SAME source cell sits at offset s_k - e_x:
//               A[i][k] = W[c][s_k] (v = 0, if s_k is in the list of the even class), W[c][s_k - e_x] (v = 1, if that
//               is in the list of the odd class), else 0.
// Siblings share their parent, hence (Eq. 15) almost all of their source cells: the union U of the two lists, in
// source-cell coordinates, is 0.1 % .. 8 % longer than either list, so 92 - 99.9 % of the multiplications are useful.
// The host lays U out in chunks of 4 offsets as a table of ready-made A fragments (one double + one tile offset per
// lane and chunk, identical for every block: read through L1), per (y, z)-parity pair.
// Block = 8 warps = a 16 x 16 x 8 target tile (two blocks per SM, so that one block's tile load hides behind the
// other's arithmetic); the masses of tile + halo arrive as one TMA box like in p2p_monopole_kernel.  A warp owns the
// 16 x-rows of one (y, z)-parity pair in two layers: per chunk it loads one A fragment and 16 B fragments (LDS.64 at
// compile-time offsets from one address) and issues 16 independent DMMAs.
// ------------------------------------------------------------------------------------------
constexpr int DT_Z = 8;
constexpr int DS_Z = DT_Z + 2 * REACH_MAX;                                   // 18 layers
constexpr int DMMA_TILE_BYTES = MS_ROW * MS_Y * DS_Z * 8;                    // 104832 B
constexpr int DMMA_SMEM = DMMA_TILE_BYTES + 64;
constexpr int DMMA_THREADS = 256;
constexpr int DMMA_MAX_CHUNKS = (2 * REACH_MAX + 2) * (2 * REACH_MAX + 1) * (2 * REACH_MAX + 1) / 4;   // |U| <= 12 * 11 * 11
static_assert(2 * DMMA_SMEM <= 227 * 1024, "two blocks per SM");

struct DmmaEntry {
    double a;      // this lane's element of the A fragment: A[lane >> 2][lane & 3]
    int off;       // tile offset (doubles) of source offset k = lane & 3, relative to the target row's base
    int pad;
};
struct DmmaLists {
    int nchunk[4];   // chunks of (py, pz) pair cp = py + 2 pz; its table starts at tab + cp * DMMA_MAX_CHUNKS * 32
};

__device__ __forceinline__ void dmma_8x8x4(double& d0, double& d1, double a, double b)
{
    asm volatile("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0, %1}, {%2}, {%3}, {%0, %1};"
                 : "+d"(d0), "+d"(d1) : "d"(a), "d"(b));
}

// Complete solve: the leaf evaluation fused into the tensor-core leaf kernels (FUSE_EVAL).  When the sums of a block
// are done its mass tile is dead, so the block parks them there, res = [NCOMP][8][16][16], and thread t takes parent cell
// (t & 7, (t >> 3) & 7, t >> 6) of the tile: it loads the parent's finished expansion once, evaluates it at the centres of
// its 8 leaves (phi += L0(e), g -= L1(e) + correction, e = ((a,b,c) - 1/2) h - delta_P) and stores every output exactly
// once as x-pairs -- what leaf_eval_kernel does in a second pass over the leaves (read + write of all outputs).
// Whole-grid output with even extents (the solver's leaves); out 16-byte aligned.
template <int NCOMP>
__device__ __forceinline__ void fused_leaf_eval(const Params& p, const double* __restrict__ res, double* __restrict__ out,
                                                int x0, int y0, int z0)
{
    const int t = threadIdx.x;
    const int I = t & 7, J = (t >> 3) & 7, K = t >> 6;
    const int gx = x0 + 2 * I, gy = y0 + 2 * J, gz = z0 + 2 * K;
    if (gx >= p.hi[0] || gy >= p.hi[1] || gz >= p.hi[2]) return;
    const int pnx = p.nx >> 1, pny = p.ny >> 1;
    const long long pcell = (long long)pnx * pny * (p.nz >> 1), ocell = (long long)p.ox * p.oy * p.oz;
    const long long P = ((long long)(gz >> 1) * pny + (gy >> 1)) * pnx + (gx >> 1);
    double L[20], C[3], dP[3];
#pragma unroll
    for (int c = 0; c < 20; ++c) L[c] = p.pL[c * pcell + P];
#pragma unroll
    for (int c = 0; c < 3; ++c) { C[c] = p.pC[c * pcell + P]; dP[c] = p.poff[c * pcell + P]; }
    const double h = p.hc;
#pragma unroll
    for (int cz = 0; cz < 2; ++cz)
#pragma unroll
        for (int cy = 0; cy < 2; ++cy) {
            const int r = ((2 * K + cz) * MT_Y + (2 * J + cy)) * MT_X + 2 * I;
            const long long o = ((long long)(gz + cz - p.lo[2]) * p.oy + (gy + cy - p.lo[1])) * p.ox + (gx - p.lo[0]);
            double sh0[20], sh1[20];
            const double e0[3] = {-0.5 * h - dP[0], ((double)cy - 0.5) * h - dP[1], ((double)cz - 0.5) * h - dP[2]};
            const double e1[3] = {0.5 * h - dP[0], e0[1], e0[2]};
            taylor_shift<1>(L, e0, sh0);
            taylor_shift<1>(L, e1, sh1);
            const double2 s = *reinterpret_cast<const double2*>(res + r);
            *reinterpret_cast<double2*>(out + o) = make_double2(s.x + sh0[0], s.y + sh1[0]);
            if constexpr (NCOMP == 4) {
#pragma unroll
                for (int c = 0; c < 3; ++c) {
                    const double2 g = *reinterpret_cast<const double2*>(res + (1 + c) * (MT_X * MT_Y * DT_Z) + r);
                    *reinterpret_cast<double2*>(out + (1 + c) * ocell + o) =
                        make_double2(g.x - (sh0[1 + c] + C[c]), g.y - (sh1[1 + c] + C[c]));
                }
            }
        }
}

template <bool FUSE_EVAL = false>
__global__ void __launch_bounds__(DMMA_THREADS, 2)
p2p_monopole_dmma_kernel(const __grid_constant__ CUtensorMap tmap, const Params p, const DmmaEntry* __restrict__ tab,
                         const DmmaLists dl, double* __restrict__ out)
{
    extern __shared__ __align__(128) unsigned char mono_smem[];
    double* tile = reinterpret_cast<double*>(mono_smem);
    uint64_t* bar = reinterpret_cast<uint64_t*>(mono_smem + DMMA_TILE_BYTES);
    const int warp = __shfl_sync(0xffffffffu, (int)(threadIdx.x >> 5), 0);
    const int lane = threadIdx.x & 31;
    const int bx = (p.ox + MT_X - 1) / MT_X, by = (p.oy + MT_Y - 1) / MT_Y;
    const int b = p.tile_list ? p.tile_list[blockIdx.x] : (int)blockIdx.x + p.tile_offset;   // tree levels: only the tiles that hold leaf cells
    const int x0 = p.lo[0] + (b % bx) * MT_X, y0 = p.lo[1] + ((b / bx) % by) * MT_Y, z0 = p.lo[2] + (b / (bx * by)) * DT_Z;

    if (threadIdx.x == 0) {
        mbar_init(bar, 1);
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
        asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
        mbar_arrive_expect_tx(bar, DMMA_TILE_BYTES);
        tma_load_tile3(tile, &tmap, bar, x0 >> 1, 2 * y0, z0);
    }
    __syncthreads();                 // barrier initialised

    const int cp = warp & 3, py = cp & 1, pz = cp >> 1, half = warp >> 2;
    // rows of this warp: y = y0 + py + 2 r (r = 0..7), z = z0 + pz + 4 half + 2 zz (zz = 0, 1)
    const double* base = tile + ((pz + 4 * half + REACH_MAX) * MS_Y + (py + REACH_MAX)) * MS_ROW + (lane >> 2);
    const int nch = cp == 0 ? dl.nchunk[0] : cp == 1 ? dl.nchunk[1] : cp == 2 ? dl.nchunk[2] : dl.nchunk[3];
    const int4* t = reinterpret_cast<const int4*>(tab + (size_t)cp * DMMA_MAX_CHUNKS * 32 + lane);
    double acc[16][2];
#pragma unroll
    for (int g = 0; g < 16; ++g) acc[g][0] = acc[g][1] = 0.0;
    int4 e = __ldg(t);
    mbar_wait(bar, 0);               // tile in place
#pragma unroll 1
    for (int c = 0; c < nch; ++c) {
        const int4 en = __ldg(t + (size_t)min(c + 1, nch - 1) * 32);       // next chunk's fragment
        const double a = __hiloint2double(e.y, e.x);
        const double* q = base + e.z;
        double m[16];
#pragma unroll
        for (int g = 0; g < 16; ++g) m[g] = q[((g >> 3) * 2 * MS_Y + (g & 7) * 2) * MS_ROW];
#pragma unroll
        for (int g = 0; g < 16; ++g) dmma_8x8x4(acc[g][0], acc[g][1], a, m[g]);
        e = en;
    }

    // D fragment: row = lane >> 2 -> component (lane >> 2) & 3, variant v = lane >> 4; columns 2 (lane & 3) + {0, 1}
    // -> cells x0 + 4 (lane & 3) + v (d0) and + 2 (d1).  One exchange with lane ^ 16 gives every lane two
    // x-consecutive cells, so that a warp stores four 128-byte row segments (one per component).
    const int v = lane >> 4, comp = (lane >> 2) & 3;
    const int gx = x0 + 4 * (lane & 3) + 2 * v;
    const long long ocell = (long long)p.ox * p.oy * p.oz;
    if constexpr (FUSE_EVAL) __syncthreads();          // every warp has finished reading the mass tile
#pragma unroll
    for (int g = 0; g < 16; ++g) {
        const double send = v ? acc[g][0] : acc[g][1];
        const double recv = __shfl_xor_sync(0xffffffffu, send, 16);
        const double lo = v ? recv : acc[g][0], hi = v ? acc[g][1] : recv;
        const int gy = y0 + py + 2 * (g & 7), k = z0 + pz + 4 * half + 2 * (g >> 3);
        if constexpr (FUSE_EVAL) {
            *reinterpret_cast<double2*>(tile + comp * (MT_X * MT_Y * DT_Z) + ((k - z0) * MT_Y + (gy - y0)) * MT_X + (gx - x0)) =
                make_double2(lo, hi);
        } else if (gy < p.hi[1] && k < p.hi[2] && gx < p.hi[0]) {
            double* dst = out + comp * ocell + ((long long)(k - p.lo[2]) * p.oy + (gy - p.lo[1])) * p.ox + (gx - p.lo[0]);
            if (gx + 1 < p.hi[0] && (reinterpret_cast<uintptr_t>(dst) & 15) == 0) {
                *reinterpret_cast<double2*>(dst) = make_double2(lo, hi);
            } else {
                dst[0] = lo;
                if (gx + 1 < p.hi[0]) dst[1] = hi;
            }
        }
    }
    if constexpr (FUSE_EVAL) {
        __syncthreads();
        fused_leaf_eval<4>(p, tile, out, x0, y0, z0);
    }
}

// ------------------------------------------------------------------------------------------
// Potential-only monopole sum for the second right-hand side of the complete solve (d(phi)/dt from d(mass)/dt,
// only the potential of that solve is used, Eq. 3), on the same tensor-core instruction.
// With one output per target the 8 rows of a DMMA are the 8 CHILDREN of one parent cell (they share the parent,
// hence -- Eq. 15 -- all source cells of the leaf list: 264 positions for 263 partners each), the 8 columns are 8
// parents next to each other in x, k runs over 4 source positions s_k relative to the parent's (even, even, even)
// child:  A[v][k] = W_phi[s_k - c_v] (0 if that offset is not in child v's list),  B[k][j] = m[t_j + s_k].
// One DMMA = 8 parents x 8 children x 4 sources, a quarter of the instructions of the four-output kernel.
// Block = 8 warps = a 16 x 16 x 8 target tile = 32 parent rows of 8 parents; a warp owns 4 of them.
// ------------------------------------------------------------------------------------------
constexpr int DMMA_MAX_CHUNKS_POT = (2 * REACH_MAX + 2) * (2 * REACH_MAX + 2) * (2 * REACH_MAX + 2) / 4;   // |U| <= 12^3

__global__ void __launch_bounds__(DMMA_THREADS, 2)
p2p_potential_dmma_kernel(const __grid_constant__ CUtensorMap tmap, const Params p, const DmmaEntry* __restrict__ tab,
                          const int nch, double* __restrict__ out)
{
    extern __shared__ __align__(128) unsigned char mono_smem[];
    double* tile = reinterpret_cast<double*>(mono_smem);
    uint64_t* bar = reinterpret_cast<uint64_t*>(mono_smem + DMMA_TILE_BYTES);
    const int warp = __shfl_sync(0xffffffffu, (int)(threadIdx.x >> 5), 0);
    const int lane = threadIdx.x & 31;
    const int bx = (p.ox + MT_X - 1) / MT_X, by = (p.oy + MT_Y - 1) / MT_Y;
    const int b = blockIdx.x;
    const int x0 = p.lo[0] + (b % bx) * MT_X, y0 = p.lo[1] + ((b / bx) % by) * MT_Y, z0 = p.lo[2] + (b / (bx * by)) * DT_Z;

    if (threadIdx.x == 0) {
        mbar_init(bar, 1);
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
        asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
        mbar_arrive_expect_tx(bar, DMMA_TILE_BYTES);
        tma_load_tile3(tile, &tmap, bar, x0 >> 1, 2 * y0, z0);
    }
    __syncthreads();

    // parent rows of this warp: y = y0 + 8 (warp & 1) + 2 i (i = 0..3), z = z0 + 2 (warp >> 1)
    const int yb = 8 * (warp & 1), zb = 2 * (warp >> 1);
    const double* base = tile + ((zb + REACH_MAX) * MS_Y + (yb + REACH_MAX)) * MS_ROW + (lane >> 2);
    const int4* t = reinterpret_cast<const int4*>(tab + lane);
    double acc[4][2];
#pragma unroll
    for (int g = 0; g < 4; ++g) acc[g][0] = acc[g][1] = 0.0;
    // the A fragments come from global memory (L1 / L2): with 4 contractions per chunk a warp has only ~64 cycles of
    // work per fragment, so the loads run POT_PREFETCH chunks ahead in a register ring
    constexpr int POT_PREFETCH = 8;
    int4 e[POT_PREFETCH];
#pragma unroll
    for (int u = 0; u < POT_PREFETCH; ++u) e[u] = __ldg(t + (size_t)min(u, nch - 1) * 32);
    mbar_wait(bar, 0);
#pragma unroll 1
    for (int c = 0; c < nch; c += POT_PREFETCH) {
#pragma unroll
        for (int u = 0; u < POT_PREFETCH; ++u) {
            if (c + u < nch) {                                  // warp-uniform
                const int4 cur = e[u];
                e[u] = __ldg(t + (size_t)min(c + u + POT_PREFETCH, nch - 1) * 32);
                const double a = __hiloint2double(cur.y, cur.x);
                const double* q = base + cur.z;
                double m[4];
#pragma unroll
                for (int g = 0; g < 4; ++g) m[g] = q[g * 2 * MS_ROW];
#pragma unroll
                for (int g = 0; g < 4; ++g) dmma_8x8x4(acc[g][0], acc[g][1], a, m[g]);
            }
        }
    }

    // D fragment: row = lane >> 2 = child v = vx + 2 vy + 4 vz; columns 2 (lane & 3) + {0, 1} = parents.
    // d0 -> cell x0 + 4 (lane & 3) + vx, d1 -> + 2.  One exchange with lane ^ 4 (the other vx) gives every lane two
    // x-consecutive cells.
    const int v = lane >> 2, vx = v & 1, vy = (v >> 1) & 1, vz = v >> 2;
    const int gx = x0 + 4 * (lane & 3) + 2 * vx;
    const int k = z0 + zb + vz;
#pragma unroll
    for (int g = 0; g < 4; ++g) {
        const double send = vx ? acc[g][0] : acc[g][1];
        const double recv = __shfl_xor_sync(0xffffffffu, send, 4);
        const double lo = vx ? recv : acc[g][0], hi = vx ? acc[g][1] : recv;
        const int gy = y0 + yb + 2 * g + vy;
        if (gy < p.hi[1] && k < p.hi[2] && gx < p.hi[0]) {
            double* dst = out + ((long long)(k - p.lo[2]) * p.oy + (gy - p.lo[1])) * p.ox + (gx - p.lo[0]);
            if (gx + 1 < p.hi[0] && (reinterpret_cast<uintptr_t>(dst) & 15) == 0) {
                *reinterpret_cast<double2*>(dst) = make_double2(lo, hi);
            } else {
                dst[0] = lo;
                if (gx + 1 < p.hi[0]) dst[1] = hi;
            }
        }
    }
}

// ------------------------------------------------------------------------------------------
// FP64 ALU roofline probe: 8 independent DFMA chains per thread.
// ------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(256) dfma_peak_kernel(double* out, int iters, double seed)
{
    double a0 = seed + threadIdx.x, a1 = a0 + 1, a2 = a0 + 2, a3 = a0 + 3, a4 = a0 + 4, a5 = a0 + 5, a6 = a0 + 6, a7 = a0 + 7;
    const double m = 0.999999, c = 1e-9;
#pragma unroll 1
    for (int i = 0; i < iters; ++i) {
#pragma unroll
        for (int u = 0; u < 8; ++u) {
            a0 = fma(a0, m, c); a1 = fma(a1, m, c); a2 = fma(a2, m, c); a3 = fma(a3, m, c);
            a4 = fma(a4, m, c); a5 = fma(a5, m, c); a6 = fma(a6, m, c); a7 = fma(a7, m, c);
        }
    }
    out[(size_t)blockIdx.x * blockDim.x + threadIdx.x] = ((a0 + a1) + (a2 + a3)) + ((a4 + a5) + (a6 + a7));
}


// FP64 issue-rate probe with register operands (the peak probe above uses immediates):
//   MODE 0: a[i] = fma(b[.], c[.], a[i]) with three fresh register operands per instruction
//   MODE 1: a[i] = fma(b[u], c[i], a[i]): 16 consecutive DFMAs repeat b[u] in the same slot (operand-reuse cache)
//   MODE 2: a[i] = a[i] * b[.]  (DMUL, two register operands)
template <int MODE>
__global__ void __launch_bounds__(384) fp64_issue_probe_kernel(double* out, const double* __restrict__ in, int iters)
{
    constexpr int NA = 16;
    double a[NA], b[4], c[8];
#pragma unroll
    for (int i = 0; i < NA; ++i) a[i] = in[threadIdx.x + i];
#pragma unroll
    for (int i = 0; i < 4; ++i) b[i] = in[64 + threadIdx.x + i];
#pragma unroll
    for (int i = 0; i < 8; ++i) c[i] = in[128 + threadIdx.x + i];
#pragma unroll 1
    for (int it = 0; it < iters; ++it) {
#pragma unroll
        for (int u = 0; u < 4; ++u)
#pragma unroll
            for (int i = 0; i < NA; ++i) {
                if (MODE == 0) a[i] = fma(b[(i + u) & 3], c[(i * 3 + u) & 7], a[i]);
                else if (MODE == 1) a[i] = fma(b[u], c[i & 7], a[i]);
                else a[i] = a[i] * b[(i + u) & 3];
            }
    }
    double s = 0.0;
#pragma unroll
    for (int i = 0; i < NA; ++i) s += a[i];
    out[(size_t)blockIdx.x * blockDim.x + threadIdx.x] = s;
}

}  // namespace octo
