// octo_fmm.cu -- C ABI (include/octo_fmm.h) and host logic of the B200-native FMM
// cell-to-cell interaction step.  Kernels live in kernels.cuh / m2l_math.cuh.
//
// Host logic here: configuration checks, the interaction lists of Eq. 15,
// their translation into shared-memory offsets, the closed-form interaction count, the TMA
// descriptor of the staged source array, workspace partitioning, launches.
#include <cuda.h>
#include <cuda_runtime.h>

#include <algorithm>
#include <cmath>
#include <cstdio>
#include <cstring>
#include <mutex>
#include <new>
#include <utility>
#include <vector>

#include "../../include/octo_fmm.h"
#include "kernels.cuh"
#include "solver.cuh"
#include "tree.cuh"

using namespace octo;

namespace {

constexpr size_t ALIGN = 256;
constexpr int MAX_CHUNKS = 32;
constexpr long long WARP_KERNEL_MAX_CELLS = 4096;   // at most this many targets: m2l_warp_kernel by default
inline size_t align_up(size_t v) { return (v + ALIGN - 1) / ALIGN * ALIGN; }

struct Offset3 { signed char d[3]; };

// Eq. 15 with distances in units of the (parent) cell width: theta' = 1/|Delta| < theta.
inline bool well_separated(long long d2, double theta) { return (double)d2 * theta * theta > 1.0; }
inline int floor_div2(int v) { return v >> 1; }   // arithmetic shift: floor for negatives too
inline int floor_div8(int v) { return v >> 3; }

// partner list of parity class (px,py,pz): cells well separated, parents not (L135)
// leaf: the leaf-level list of the complete solve -- every Delta != 0 whose parents are not well separated
// (the Eq. 15 list plus the near field)
std::vector<Offset3> build_list(int px, int py, int pz, double theta, int* reach_out, bool leaf = false)
{
    std::vector<Offset3> out;
    const int S = 2 * (int)std::floor(1.0 / theta) + 3;
    int reach = 0;
    for (int dz = -S; dz <= S; ++dz)
        for (int dy = -S; dy <= S; ++dy)
            for (int dx = -S; dx <= S; ++dx) {
                const long long c2 = (long long)dx * dx + (long long)dy * dy + (long long)dz * dz;
                if (c2 == 0 || (!leaf && !well_separated(c2, theta))) continue;
                const int Ix = floor_div2(px + dx), Iy = floor_div2(py + dy), Iz = floor_div2(pz + dz);
                const long long p2 = (long long)Ix * Ix + (long long)Iy * Iy + (long long)Iz * Iz;
                if (p2 != 0 && well_separated(p2, theta)) continue;
                Offset3 o;
                o.d[0] = (signed char)dx; o.d[1] = (signed char)dy; o.d[2] = (signed char)dz;
                out.push_back(o);
                const int m = std::max(std::abs(dx), std::max(std::abs(dy), std::abs(dz)));
                if (m > reach) reach = m;
            }
    if (reach_out && reach > *reach_out) *reach_out = reach;
    return out;
}

// creation flags of internal handles (the levels of the complete solve)
constexpr int CF_ANY_SIZE = 1;    // any even grid size >= 2 (whole-grid output); sizes that are not multiples of 8 use the direct kernel
constexpr int CF_LEAF_LIST = 2;   // monopole kind with the leaf-level list (Eq. 15 list + near field)

bool region_of(const octo_fmm_config& c, int lo[3], int hi[3], int flags = 0)
{
    bool whole = true;
    for (int a = 0; a < 3; ++a) whole = whole && c.out_lo[a] == 0 && c.out_hi[a] == 0;
    for (int a = 0; a < 3; ++a) {
        lo[a] = whole ? 0 : c.out_lo[a];
        hi[a] = whole ? c.n[a] : c.out_hi[a];
        if (lo[a] < 0 || hi[a] > c.n[a] || lo[a] >= hi[a]) return false;
        if (!(flags & CF_ANY_SIZE) && (lo[a] % 8 || hi[a] % 8)) return false;
    }
    return true;
}

bool config_ok(const octo_fmm_config* c, int flags = 0)
{
    if (!c) return false;
    for (int a = 0; a < 3; ++a)
        if (c->n[a] <= 0 || c->n[a] % ((flags & CF_ANY_SIZE) ? 2 : 8) || c->n[a] > 4096) return false;
    int lo[3], hi[3];
    if (!region_of(*c, lo, hi, flags)) return false;
    if (!(c->h > 0.0) || !std::isfinite(c->h)) return false;
    if (!(c->theta > 1.0 / 3.0 && c->theta < 1.0)) return false;   // reach <= 5 (theta_min, L137)
    if (c->kind != OCTO_FMM_MULTIPOLE && c->kind != OCTO_FMM_MONOPOLE) return false;
    return true;
}

struct Sizes { size_t src, L, C, W, T, flags, total; };

Sizes sizes_of(const octo_fmm_config& c, int flags = 0)
{
    int lo[3], hi[3];
    region_of(c, lo, hi, flags);
    const size_t ncell = (size_t)c.n[0] * c.n[1] * c.n[2];
    const size_t ocell = (size_t)(hi[0] - lo[0]) * (hi[1] - lo[1]) * (hi[2] - lo[2]);
    Sizes s{};
    if (c.kind == OCTO_FMM_MULTIPOLE) {
        s.src = align_up(ncell * NPAIR * 2 * sizeof(double));
        s.L = align_up(ocell * 20 * sizeof(double));
        s.C = align_up(ocell * 3 * sizeof(double));
    } else {
        const size_t pc = (size_t)(c.n[0] + REACH_MAX + MONO_PAD_RIGHT) * (c.n[1] + 2 * REACH_MAX) * (c.n[2] + 2 * REACH_MAX);
        s.src = align_up(pc * sizeof(double));
        s.L = align_up(ocell * 4 * sizeof(double));
        s.C = 0;
        s.W = align_up((size_t)MONO_NW * sizeof(double4));
        s.T = align_up(((size_t)4 * DMMA_MAX_CHUNKS + DMMA_MAX_CHUNKS_POT) * 32 * sizeof(DmmaEntry));
    }
    s.flags = ALIGN;
    s.total = s.src + s.L + s.C + s.W + s.T + s.flags;
    return s;
}

typedef CUresult (*EncodeTiledFn)(CUtensorMap*, CUtensorMapDataType, cuuint32_t, void*, const cuuint64_t*,
                                  const cuuint64_t*, const cuuint32_t*, const cuuint32_t*, CUtensorMapInterleave,
                                  CUtensorMapSwizzle, CUtensorMapL2promotion, CUtensorMapFloatOOBfill);

EncodeTiledFn encode_tiled_fn()
{
    static EncodeTiledFn fn = nullptr;
    if (!fn) {
        void* p = nullptr;
        cudaDriverEntryPointQueryResult q;
        if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &p, cudaEnableDefault, &q) == cudaSuccess &&
            q == cudaDriverEntryPointSuccess)
            fn = (EncodeTiledFn)p;
    }
    return fn;
}

// One row of the 8 x 4 A fragment of the tensor-core monopole kernels: the outputs of this row belong to the target
// shifted by (cx, cy, cz) from the base target, whose interaction list is *list, and are component comp of the weights.
struct DmmaRow { const std::vector<Offset3>* list; int cx, cy, cz, comp; };

// Table of A fragments, one chunk = 4 source positions relative to the base target.  U = the union over the rows of
// (list + shift), in (sz, sy, sx) order.  A[i][k] = weight comp_i of offset (s_k - shift_i) if that offset is in row i's
// list, else 0.  The 4 positions of a chunk are chosen so that the B-fragment load (kernels.cuh) has no shared-memory
// bank conflict: an LDS.64 is served per half-warp = 4 targets (j) x 4 positions (k) at addresses off_k + j; two
// positions are compatible if their 4-double segments overlap in ADDRESS (|difference| <= 3: broadcast) or lie at least
// 4 banks (of 8 bytes, 16 per 128-byte wavefront) apart.  Greedy in list order; a slot left empty repeats the chunk's
// first position with zero weights.  Returns the number of chunks, -1 if they exceed max_chunks.
int build_dmma_table(const DmmaRow (&rows)[8], const std::vector<double4>& wt, DmmaEntry* tb, int max_chunks)
{
    constexpr int NP = 2 * REACH_MAX + 2;     // positions -5 .. 6 per axis
    auto pos = [&](int sx, int sy, int sz) { return ((size_t)(sz + REACH_MAX) * NP + (sy + REACH_MAX)) * NP + (sx + REACH_MAX); };
    auto widx_of = [](int dx, int dy, int dz) {
        return ((dz + REACH_MAX) * (2 * REACH_MAX + 1) + (dy + REACH_MAX)) * (2 * REACH_MAX + 1) + (dx + REACH_MAX);
    };
    std::vector<unsigned char> in((size_t)NP * NP * NP, 0);      // bit i: position is in row i's shifted list
    for (int i = 0; i < 8; ++i)
        for (const Offset3& o : *rows[i].list) in[pos(o.d[0] + rows[i].cx, o.d[1] + rows[i].cy, o.d[2] + rows[i].cz)] |= (unsigned char)(1u << i);
    struct Src { int sx, sy, sz, off; unsigned char rows; };
    std::vector<Src> U;
    for (int sz = -REACH_MAX; sz <= REACH_MAX + 1; ++sz)
        for (int sy = -REACH_MAX; sy <= REACH_MAX + 1; ++sy)
            for (int sx = -REACH_MAX; sx <= REACH_MAX + 1; ++sx) {
                const unsigned char r = in[pos(sx, sy, sz)];
                if (!r) continue;
                const int off = (sz * MS_Y + sy) * MS_ROW + (((sx + REACH_MAX) & 1) ? MS_XH : 0) + ((sx + REACH_MAX) >> 1);
                U.push_back(Src{sx, sy, sz, off, r});
            }
    auto compatible = [](int a, int b) {
        const int d = b - a;
        if (d >= -3 && d <= 3) return true;
        const int D = ((d % 16) + 16) % 16;
        return D >= 4 && D <= 12;
    };
    std::vector<char> used(U.size(), 0);
    int nchunk = 0;
    for (size_t first = 0; first < U.size(); ++first) {
        if (used[first]) continue;
        if (nchunk == max_chunks) return -1;
        size_t member[4];
        int nm = 0;
        member[nm++] = first; used[first] = 1;
        for (size_t j = first + 1; j < U.size() && nm < 4; ++j) {
            if (used[j]) continue;
            bool ok = true;
            for (int k = 0; k < nm; ++k) ok = ok && compatible(U[member[k]].off, U[j].off);
            if (ok) { member[nm++] = j; used[j] = 1; }
        }
        for (int k = 0; k < 4; ++k) {
            const Src* u = k < nm ? &U[member[k]] : nullptr;
            for (int i = 0; i < 8; ++i) {
                DmmaEntry& t = tb[(size_t)nchunk * 32 + 4 * i + k];
                t.off = u ? u->off : U[first].off;
                double w = 0.0;
                if (u && ((u->rows >> i) & 1)) {
                    const double4& q = wt[widx_of(u->sx - rows[i].cx, u->sy - rows[i].cy, u->sz - rows[i].cz)];
                    const int c = rows[i].comp;
                    w = c == 0 ? q.x : c == 1 ? q.y : c == 2 ? q.z : q.w;
                }
                t.a = w;
            }
        }
        ++nchunk;
    }
    return nchunk;
}

// Monopole weights of the 11^3 offsets: (-1/|R|, -R/|R|^3) with R = (i_A - i_B) h = -Delta h (hmul[d + 5] = -d h), in
// FP64 on the host (sqrt, division); Delta = 0 gets zero weights.
std::vector<double4> monopole_weights(const double (&hmul)[2 * REACH_MAX + 1])
{
    std::vector<double4> wt((size_t)MONO_NW, double4{0.0, 0.0, 0.0, 0.0});
    for (int dz = -REACH_MAX; dz <= REACH_MAX; ++dz)
        for (int dy = -REACH_MAX; dy <= REACH_MAX; ++dy)
            for (int dx = -REACH_MAX; dx <= REACH_MAX; ++dx) {
                if (!dx && !dy && !dz) continue;
                const double Rx = hmul[dx + REACH_MAX], Ry = hmul[dy + REACH_MAX], Rz = hmul[dz + REACH_MAX];
                const double r2 = Rx * Rx + Ry * Ry + Rz * Rz, r = std::sqrt(r2), ir3 = -1.0 / (r2 * r);
                const int widx = ((dz + REACH_MAX) * (2 * REACH_MAX + 1) + (dy + REACH_MAX)) * (2 * REACH_MAX + 1) + (dx + REACH_MAX);
                wt[widx] = double4{-1.0 / r, Rx * ir3, Ry * ir3, Rz * ir3};
            }
    return wt;
}

// The rows of the two tensor-core tables: which = 0..3 -> p2p_monopole_dmma_kernel for (py, pz) = (which & 1, which >> 1):
// rows 0-3 = (phi, g) of the x-even target, rows 4-7 of its x-odd sibling; which = 4 -> p2p_potential_dmma_kernel: row v =
// the potential of child v = vx + 2 vy + 4 vz of one parent.
void dmma_rows(const std::vector<Offset3> (&list)[8], int which, DmmaRow (&rows)[8])
{
    for (int i = 0; i < 8; ++i) {
        if (which < 4) rows[i] = DmmaRow{&list[(i >> 2) + 2 * (which & 1) + 4 * (which >> 1)], i >> 2, 0, 0, i & 3};
        else           rows[i] = DmmaRow{&list[i], i & 1, (i >> 1) & 1, i >> 2, 0};
    }
}

// The interaction lists live in ONE __constant__ bank per device (kernels.cuh: c_entries, c_begin, c_near): they depend
// on (theta, kind, list flavour) only, so the levels of a complete solve and every handle with the same theta share them
// and nothing is uploaded in the steady state.  Handles with DIFFERENT lists may be driven from different streams and
// host threads; the bank serialises them: a host mutex guards the book-keeping, every kernel that reads the bank leaves
// an event on its stream, and an upload first makes its stream wait for the readers of the previous contents on other
// streams (and a reader on another stream waits for the upload).  Everything that depends on a handle's h is in Params.
constexpr int MAX_DEVICES = 64;
struct ConstBank {
    std::mutex mu;
    unsigned long long sig = 0;                               // lists in (or on their way into) the bank
    cudaStream_t up_stream = nullptr;                         // stream the current contents were uploaded on
    cudaEvent_t uploaded = nullptr;                           // recorded after that upload
    std::vector<std::pair<cudaStream_t, cudaEvent_t>> readers;   // last reading kernel of every stream since the upload
    std::vector<cudaEvent_t> pool;                            // spare events
};
ConstBank g_bank[MAX_DEVICES];

}  // namespace

struct octo_fmm {
    octo_fmm_config cfg;
    int lo[3], hi[3];
    int reach;
    std::vector<Offset3> list[8];
    std::vector<StEntry> entries;          // 8 * MAX_LIST
    std::vector<char4> near_list;          // 8 * MAX_NEAR: the near field of each parity class (mixed levels, f3)
    std::vector<StEntry> entries_mixed;    // 8 * MAX_LIST: Eq. 15 list + near field (d2 = 1 marks a near-field entry), staged kernel
    int begin_mixed[8][2 * REACH_MAX + 2];
    unsigned long long list_sig_mixed;
    int mixed_count;       // 1: interact_mixed also counts its pairs (option "mixed_count")
    bool mixed_counted;    // the last interact_mixed did
    int near_count[8];
    int begin[8][2 * REACH_MAX + 2];
    double hmul[2 * REACH_MAX + 1];
    double4* W;            // monopole: device table of the weights of the 11^3 offsets
    DmmaEntry* T;          // monopole: device table of the A fragments of p2p_monopole_dmma_kernel
    DmmaLists dl;
    int nchunk_pot;        // chunks of the potential-only table (after the four tables of dl in T)
    CUtensorMap tmap2;     // monopole: the 16 x 16 x 8 tile box of p2p_monopole_dmma_kernel
    int mono_kernel;       // 0 tensor-core instruction (default), 1 DFMA
    bool mixed;            // the last interaction was octo_fmm_interact_mixed
    unsigned long long n_interactions;
    CUtensorMap tmap;      // monopole: the mass tile box of p2p_monopole_kernel
    SlabMaps maps;         // multipole: own staged array (+ the neighbours' with octo_fmm_set_neighbours)
    bool has_neighbours;
    Params prm;
    double* src;
    double* L;             // workspace result buffers
    double* C;
    double* outL;          // where interact() writes: the workspace, or the caller's bound buffers
    double* outC;
    double* resL;          // where the last interact() left its results
    double* resC;
    int* flags;
    int state;          // 0 created, 1 sources staged, 2 interacted
    int kernel;         // 0 staged (TMA), 1 direct
    int sm_count;
    cudaStream_t stream;
    // run_host pipeline (created on first use)
    unsigned long long list_sig;   // identifies the contents of entries/begin (see bank_acquire)
    int host_chunk;        // output z-layers per pipeline slab; 0 = no pipelining
    int host_launches;     // kernels the last run_host launched
    // a level of the adaptive tree solve (tree.inl): the kinds of its cells, and the bricks / tiles that have work
    const unsigned char* tree_kind;   // device [n^3]; non-null: the slab-fed kernel runs in MODE_TREE
    const int* tile_list;             // device; null = every brick (multipole) / tile (monopole)
    const unsigned short* tile_zmask; // device, per listed brick (multipole, tree levels): source layers worth loading; null = all
    int tile_count;
    int mono_zt_begin, mono_zt_end;   // tensor-core monopole kernels: z-tiles [begin, end) of this launch; end = 0: all
    int* pinned_flag;      // pinned host word the host entry points read the device flag through (no pageable copy)
    bool pipeline_ready;   // the side streams and events below all exist
    cudaStream_t s_h2d, s_d2h;
    cudaEvent_t ev_in[32], ev_out[32], ev_begin, ev_end;
};

extern "C" {

const char* octo_fmm_version(void) { return "octo_fmm 0.3 (sm_100a)"; }

size_t octo_fmm_workspace_bytes(const octo_fmm_config* cfg)
{
    if (!config_ok(cfg)) return 0;
    return sizes_of(*cfg).total;
}

size_t octo_fmm_host_scratch_bytes(const octo_fmm_config* cfg)
{
    if (!config_ok(cfg)) return 0;
    int lo[3], hi[3];
    region_of(*cfg, lo, hi);
    const size_t ncell = (size_t)cfg->n[0] * cfg->n[1] * cfg->n[2];
    const size_t ocell = (size_t)(hi[0] - lo[0]) * (hi[1] - lo[1]) * (hi[2] - lo[2]);
    if (cfg->kind == OCTO_FMM_MULTIPOLE)
        return align_up(ncell * 20 * 8) + align_up(ncell * 3 * 8) + align_up(ocell * 20 * 8) + align_up(ocell * 3 * 8);
    return align_up(ncell * 8) + align_up(ocell * 4 * 8);
}

// interaction count: per-axis closed form over the lists; partners outside the grid are skipped, where the grid's
// z-extent is [zmin, zmax] (beyond [0, nz) with neighbouring z-slabs, octo_fmm_set_neighbours)
static unsigned long long count_interactions(const octo_fmm* h, int zmin, int zmax)
{
    unsigned long long cnt[3][2][2 * REACH_MAX + 1];
    for (int a = 0; a < 3; ++a) {
        const int amin = a == 2 ? zmin : 0, amax = a == 2 ? zmax : h->cfg.n[a] - 1;
        for (int par = 0; par < 2; ++par)
            for (int d = -REACH_MAX; d <= REACH_MAX; ++d) {
                unsigned long long c = 0;
                for (int i = h->lo[a]; i < h->hi[a]; ++i)
                    if ((i & 1) == par && i + d >= amin && i + d <= amax) ++c;
                cnt[a][par][d + REACH_MAX] = c;
            }
    }
    unsigned long long total = 0;
    for (int p = 0; p < 8; ++p)
        for (const Offset3& o : h->list[p])
            total += cnt[0][p & 1][o.d[0] + REACH_MAX] * cnt[1][(p >> 1) & 1][o.d[1] + REACH_MAX] *
                     cnt[2][(p >> 2) & 1][o.d[2] + REACH_MAX];
    return total;
}

// TMA descriptor of a staged multipole array S[z][cp][y][xpar][xh][2]; tensor dims (fastest first):
//      {2 (pair), nx/2 (xh), 2 ny (y*2 + xpar), 10 (cp), nz}
static int encode_slab_map(CUtensorMap* map, const double* S, int nx, int ny, int nz)
{
    EncodeTiledFn enc = encode_tiled_fn();
    if (!enc) return OCTO_FMM_ECUDA;
    const cuuint64_t nxh = (cuuint64_t)nx / 2, nxy = (cuuint64_t)nx * ny;
    cuuint64_t dims[5] = {2, nxh, 2 * (cuuint64_t)ny, (cuuint64_t)NPAIR, (cuuint64_t)nz};
    cuuint64_t strides[4] = {16, nxh * 16, nxy * 16, nxy * 16 * NPAIR};
    cuuint32_t box[5] = {2, SLAB_XH, 2 * SLAB_Y, NPAIR, 1};
    cuuint32_t estr[5] = {1, 1, 1, 1, 1};
    std::memset(map, 0, sizeof(*map));
    const CUresult r = enc(map, CU_TENSOR_MAP_DATA_TYPE_FLOAT64, 5, (void*)S, dims, strides, box, estr, CU_TENSOR_MAP_INTERLEAVE_NONE,
                           CU_TENSOR_MAP_SWIZZLE_NONE, CU_TENSOR_MAP_L2_PROMOTION_L2_128B, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
    return r == CUDA_SUCCESS ? OCTO_FMM_OK : OCTO_FMM_ECUDA;
}

static int create_internal(const octo_fmm_config* cfg, int flags, octo_fmm_t** out)
{
    if (!out) return OCTO_FMM_EINVAL;
    *out = nullptr;
    if (!config_ok(cfg, flags)) return OCTO_FMM_EINVAL;
    const Sizes sz = sizes_of(*cfg, flags);
    if (!cfg->workspace || cfg->workspace_bytes < sz.total || ((uintptr_t)cfg->workspace % ALIGN)) return OCTO_FMM_EINVAL;

    int ndev = 0;
    if (cudaGetDeviceCount(&ndev) != cudaSuccess || cfg->device < 0 || cfg->device >= ndev || cfg->device >= MAX_DEVICES) return OCTO_FMM_ECUDA;
    if (cudaSetDevice(cfg->device) != cudaSuccess) return OCTO_FMM_ECUDA;
    cudaDeviceProp prop;
    if (cudaGetDeviceProperties(&prop, cfg->device) != cudaSuccess) return OCTO_FMM_ECUDA;
    if (prop.major != 10) return OCTO_FMM_ECUDA;   // sm_100a only

    octo_fmm* h = new (std::nothrow) octo_fmm();
    if (!h) return OCTO_FMM_ENOMEM;
    h->cfg = *cfg;
    h->stream = (cudaStream_t)cfg->stream;
    h->sm_count = prop.multiProcessorCount;
    h->state = 0;
    h->kernel = 0;
    h->mono_kernel = 0;
    h->mixed = false;
    h->mixed_count = 0;
    h->mixed_counted = false;
    h->host_chunk = 12;
    h->host_launches = 0;
    h->tree_kind = nullptr; h->tile_list = nullptr; h->tile_count = 0; h->tile_zmask = nullptr;
    h->mono_zt_begin = 0; h->mono_zt_end = 0; h->pinned_flag = nullptr;
    h->pipeline_ready = false;
    h->s_h2d = nullptr; h->s_d2h = nullptr;
    for (int i = 0; i < MAX_CHUNKS; ++i) { h->ev_in[i] = nullptr; h->ev_out[i] = nullptr; }
    h->ev_begin = nullptr; h->ev_end = nullptr;
    region_of(*cfg, h->lo, h->hi, flags);
    const bool small = cfg->n[0] % 8 || cfg->n[1] % 8 || cfg->n[2] % 8;    // only with CF_ANY_SIZE
    if (small) h->kernel = 1;
    // few targets (coarse levels of the complete solve, single sub-grids): one warp per cell
    if ((long long)(h->hi[0] - h->lo[0]) * (h->hi[1] - h->lo[1]) * (h->hi[2] - h->lo[2]) <= WARP_KERNEL_MAX_CELLS) h->kernel = 2;

    // ---- a1: interaction lists (Eq. 15) ----
    h->reach = 0;
    for (int p = 0; p < 8; ++p)
        h->list[p] = build_list(p & 1, (p >> 1) & 1, (p >> 2) & 1, cfg->theta, &h->reach, (flags & CF_LEAF_LIST) != 0);
    if (h->reach > REACH_MAX) { delete h; return OCTO_FMM_EINVAL; }
    for (int p = 0; p < 8; ++p)
        if ((int)h->list[p].size() > MAX_LIST) { delete h; return OCTO_FMM_EINVAL; }

    // near field = the leaf-level list minus the Eq. 15 list (cells that are not well separated whose parents are not either)
    h->near_list.assign((size_t)8 * MAX_NEAR, char4{0, 0, 0, 0});
    for (int p = 0; p < 8; ++p) {
        int r = 0;
        const std::vector<Offset3> full = build_list(p & 1, (p >> 1) & 1, (p >> 2) & 1, cfg->theta, &r, true);
        int n = 0;
        for (const Offset3& o : full) {
            const long long c2 = (long long)o.d[0] * o.d[0] + (long long)o.d[1] * o.d[1] + (long long)o.d[2] * o.d[2];
            if (well_separated(c2, cfg->theta)) continue;
            if (n == MAX_NEAR) { delete h; return OCTO_FMM_EINVAL; }
            h->near_list[(size_t)p * MAX_NEAR + n++] = char4{o.d[0], o.d[1], o.d[2], 0};
        }
        h->near_count[p] = n;
        // the same list for the slab-fed kernel: (dz, dy, dx) order, shared-memory offsets, near-field entries marked
        if (cfg->kind == OCTO_FMM_MULTIPOLE) {
            if (p == 0) h->entries_mixed.assign((size_t)8 * MAX_LIST, StEntry{0, 0, 0, 0, 0});
            if ((int)full.size() > MAX_LIST || r > REACH_MAX) { delete h; return OCTO_FMM_EINVAL; }
            const int px = p & 1, py = (p >> 1) & 1;
            int cur = 0;
            for (int dz = -REACH_MAX; dz <= REACH_MAX + 1; ++dz) {
                while (cur < (int)full.size() && full[cur].d[2] < dz) ++cur;
                h->begin_mixed[p][dz + REACH_MAX] = cur;
            }
            for (size_t s2 = 0; s2 < full.size(); ++s2) {
                const int dx = full[s2].d[0], dy = full[s2].d[1], dz = full[s2].d[2];
                StEntry e;
                e.off = ((py + dy + REACH_MAX) * SLAB_ROW + (((px + dx) & 1) ? SLAB_XH : 0) + ((px + dx + 6) >> 1)) * 16;   // bytes
                e.dx = (signed char)(8 * dx); e.dy = (signed char)(8 * dy); e.dz = (signed char)(8 * dz);
                e.d2 = well_separated((long long)dx * dx + (long long)dy * dy + (long long)dz * dz, cfg->theta) ? 0 : 1;
                h->entries_mixed[(size_t)p * MAX_LIST + s2] = e;
            }
        }
    }

    h->entries.assign((size_t)8 * MAX_LIST, StEntry{0, 0, 0, 0, 0});
    for (int p = 0; p < 8; ++p) {
        const int px = p & 1, py = (p >> 1) & 1;
        int cur = 0;
        for (int dz = -REACH_MAX; dz <= REACH_MAX + 1; ++dz) {
            // lists are (dz,dy,dx)-lexicographic, so each dz is a contiguous range
            while (cur < (int)h->list[p].size() && h->list[p][cur].d[2] < dz) ++cur;
            h->begin[p][dz + REACH_MAX] = cur;
        }
        for (size_t s = 0; s < h->list[p].size(); ++s) {
            const int dx = h->list[p][s].d[0], dy = h->list[p][s].d[1], dz = h->list[p][s].d[2];
            StEntry e;
            // shared-memory offset of the source relative to the thread's base (see kernels.cuh)
            if (cfg->kind == OCTO_FMM_MULTIPOLE) {
                e.off = ((py + dy + REACH_MAX) * SLAB_ROW + (((px + dx) & 1) ? SLAB_XH : 0) + ((px + dx + 6) >> 1)) * 16;   // bytes
                e.dx = (signed char)(8 * dx); e.dy = (signed char)(8 * dy); e.dz = (signed char)(8 * dz);      // see StEntry
                // which sub-grids (8 cells per axis) the partners of a warp's targets fall into, relative to the targets'
                // own: a warp holds the 4 x 4 cells of one parity class of one sub-grid (twice), cell c = p + 2 j, so the
                // partner c + d lies in sub-grid floor((p + d + 2 j) / 8) in {-1, 0, 1}.  Bits 0-2: x, bits 3-5: y
                // (the levels of the adaptive tree skip entries whose partner sub-grids hold nothing to meet)
                int xm = 0, ym = 0;
                for (int j = 0; j < 4; ++j) {
                    xm |= 1 << (floor_div8(px + dx + 2 * j) + 1);
                    ym |= 1 << (floor_div8(py + dy + 2 * j) + 1);
                }
                e.d2 = (signed char)(xm | (ym << 3));
            } else {
                // monopole: offset in the de-interleaved mass tile (doubles, low 16 bits) and index of the offset's
                // weights (high 16 bits), see p2p_monopole_kernel
                const int toff = (dz * MS_Y + dy) * MS_ROW + (((px + dx + REACH_MAX) & 1) ? MS_XH : 0) + ((px + dx + REACH_MAX) >> 1);
                const int widx = ((dz + REACH_MAX) * (2 * REACH_MAX + 1) + (dy + REACH_MAX)) * (2 * REACH_MAX + 1) + (dx + REACH_MAX);
                e.off = (toff & 0xffff) | (widx << 16);
                e.d2 = (signed char)(dx * dx + dy * dy + dz * dz);
                e.dx = (signed char)dx; e.dy = (signed char)dy; e.dz = (signed char)dz;
            }
            h->entries[(size_t)p * MAX_LIST + s] = e;
        }
    }
    for (int d = -REACH_MAX; d <= REACH_MAX; ++d) h->hmul[d + REACH_MAX] = (double)(-d) * cfg->h;
    {
        unsigned long long tb;
        std::memcpy(&tb, &cfg->theta, sizeof tb);
        h->list_sig = (tb * 0x9E3779B97F4A7C15ull) ^ ((unsigned long long)(cfg->kind + 1) << 8) ^ ((unsigned long long)((flags & CF_LEAF_LIST) ? 2 : 1) << 4) ^
                      (unsigned long long)(cfg->device + 1);
        if (h->list_sig == 0) h->list_sig = 1;
        h->list_sig_mixed = h->list_sig ^ 0x5bd1e995ull;
        if (h->list_sig_mixed == 0) h->list_sig_mixed = 2;
    }

    h->has_neighbours = false;
    h->n_interactions = count_interactions(h, 0, cfg->n[2] - 1);

    // ---- workspace partition ----
    char* w = (char*)cfg->workspace;
    h->src = (double*)w; w += sz.src;
    h->L = (double*)w;   w += sz.L;
    h->C = (double*)w;   w += sz.C;
    h->W = (double4*)w;  w += sz.W;
    h->T = (DmmaEntry*)w; w += sz.T;
    h->flags = (int*)w;

    Params& P = h->prm;
    P.nx = cfg->n[0]; P.ny = cfg->n[1]; P.nz = cfg->n[2];
    for (int a = 0; a < 3; ++a) { P.lo[a] = h->lo[a]; P.hi[a] = h->hi[a]; }
    P.ox = h->hi[0] - h->lo[0]; P.oy = h->hi[1] - h->lo[1]; P.oz = h->hi[2] - h->lo[2];
    P.tiles_x = (P.ox + TILE_X - 1) / TILE_X; P.tiles_y = (P.oy + TILE_Y - 1) / TILE_Y;
    P.kb = h->lo[2]; P.ke = h->hi[2];
    P.tiles_z = (P.oz + TILE_Z - 1) / TILE_Z;
    P.ntiles = (long long)P.tiles_x * P.tiles_y * P.tiles_z;
    P.reach = h->reach;
    h->outL = h->L; h->outC = h->C;
    P.S = h->src; P.L = h->L; P.C = h->C; P.flags = h->flags;
    P.force_dipole = 0;
    P.pL = nullptr; P.pC = nullptr; P.poff = nullptr; P.hc = cfg->h;
    P.leaf = nullptr;
    P.tile_list = nullptr;
    P.tile_zmask = nullptr;
    P.tile_offset = 0;
    for (int a = 0; a < 3; ++a) { P.pdim[a] = cfg->n[a] / 2; P.psh[a] = 0; }
    for (int d = 0; d <= 2 * REACH_MAX; ++d) P.hmul[d] = h->hmul[d];
    P.zmin = 0; P.zmax = cfg->n[2] - 1; P.nz_below = 0;
    for (int pz = 0; pz < 2; ++pz) {       // dz-extent of the lists (Eq. 15 list and leaf-level list) per z-parity of the target
        int lo = REACH_MAX, hi = -REACH_MAX;
        for (int c = 4 * pz; c < 4 * pz + 4; ++c)
            for (int dz = -REACH_MAX; dz <= REACH_MAX; ++dz) {
                const bool any = h->begin[c][dz + REACH_MAX + 1] > h->begin[c][dz + REACH_MAX] ||
                                 (cfg->kind == OCTO_FMM_MULTIPOLE && h->begin_mixed[c][dz + REACH_MAX + 1] > h->begin_mixed[c][dz + REACH_MAX]);
                if (any) { lo = std::min(lo, dz); hi = std::max(hi, dz); }
            }
        if (lo > hi) { lo = 0; hi = 0; }
        P.zr[pz][0] = lo; P.zr[pz][1] = hi;
    }
    P.nflags[0] = nullptr; P.nflags[1] = nullptr;

    if (cfg->kind == OCTO_FMM_MULTIPOLE && !small) {
        if (encode_slab_map(&h->maps.own, h->src, cfg->n[0], cfg->n[1], cfg->n[2]) != OCTO_FMM_OK) { delete h; return OCTO_FMM_ECUDA; }
        h->maps.below = h->maps.own; h->maps.above = h->maps.own;
        cudaError_t e1 = cudaFuncSetAttribute(m2l_staged_kernel<true>, cudaFuncAttributeMaxDynamicSharedMemorySize, STAGED_SMEM);
        cudaError_t e2 = cudaFuncSetAttribute(m2l_staged_kernel<false>, cudaFuncAttributeMaxDynamicSharedMemorySize, STAGED_SMEM);
        cudaError_t e3 = cudaFuncSetAttribute(m2l_staged_kernel<true, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, STAGED_SMEM);
        cudaError_t e4 = cudaFuncSetAttribute(m2l_staged_kernel<false, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, STAGED_SMEM);
        cudaError_t e5 = cudaFuncSetAttribute(m2l_staged_kernel<true, false, MODE_MIXED>, cudaFuncAttributeMaxDynamicSharedMemorySize, STAGED_SMEM);
        cudaError_t e6 = cudaFuncSetAttribute(m2l_staged_kernel<false, false, MODE_MIXED>, cudaFuncAttributeMaxDynamicSharedMemorySize, STAGED_SMEM);
        cudaError_t e7 = cudaFuncSetAttribute(m2l_staged_kernel<true, true, MODE_TREE>, cudaFuncAttributeMaxDynamicSharedMemorySize, STAGED_SMEM);
        cudaError_t e8 = cudaFuncSetAttribute(m2l_staged_kernel<false, true, MODE_TREE>, cudaFuncAttributeMaxDynamicSharedMemorySize, STAGED_SMEM);
        if (cudaFuncSetAttribute(m2l_staged_kernel<true, false, MODE_TREE>, cudaFuncAttributeMaxDynamicSharedMemorySize, STAGED_SMEM) != cudaSuccess ||
            cudaFuncSetAttribute(m2l_staged_kernel<false, false, MODE_TREE>, cudaFuncAttributeMaxDynamicSharedMemorySize, STAGED_SMEM) != cudaSuccess) {
            delete h; return OCTO_FMM_ECUDA;
        }
        if (e1 != cudaSuccess || e2 != cudaSuccess || e3 != cudaSuccess || e4 != cudaSuccess || e5 != cudaSuccess || e6 != cudaSuccess ||
            e7 != cudaSuccess || e8 != cudaSuccess) {
            delete h; return OCTO_FMM_ECUDA;
        }
    } else if (cfg->kind == OCTO_FMM_MONOPOLE) {
        // ---- monopole weights of the 11^3 offsets: (-1/|R|, -R/|R|^3) with R = (i_A - i_B) h = -Delta h, in FP64
        //      on the host (sqrt, division); Delta = 0 gets zero weights ----
        const std::vector<double4> wt = monopole_weights(h->hmul);
        if (cudaMemcpyAsync(h->W, wt.data(), wt.size() * sizeof(double4), cudaMemcpyHostToDevice, h->stream) != cudaSuccess ||
            cudaStreamSynchronize(h->stream) != cudaSuccess) { delete h; return OCTO_FMM_ECUDA; }
        // ---- TMA descriptor of the staged masses P[z][y * 2 + xpar][xh] (see stage_monopole_kernel) ----
        EncodeTiledFn enc = encode_tiled_fn();
        if (!enc) { delete h; return OCTO_FMM_ECUDA; }
        const cuuint64_t X = (cuuint64_t)cfg->n[0] + REACH_MAX + MONO_PAD_RIGHT, Y = (cuuint64_t)cfg->n[1] + 2 * REACH_MAX,
                         Z = (cuuint64_t)cfg->n[2] + 2 * REACH_MAX;
        cuuint64_t mdims[3] = {X / 2, 2 * Y, Z};
        cuuint64_t mstrides[2] = {X / 2 * 8, X * Y * 8};
        cuuint32_t mbox[3] = {MS_XH, 2 * MS_Y, MS_Z};
        cuuint32_t mestr[3] = {1, 1, 1};
        std::memset(&h->tmap, 0, sizeof(h->tmap));
        if (enc(&h->tmap, CU_TENSOR_MAP_DATA_TYPE_FLOAT64, 3, (void*)h->src, mdims, mstrides, mbox, mestr, CU_TENSOR_MAP_INTERLEAVE_NONE,
                CU_TENSOR_MAP_SWIZZLE_NONE, CU_TENSOR_MAP_L2_PROMOTION_L2_128B, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE) != CUDA_SUCCESS) {
            delete h; return OCTO_FMM_ECUDA;
        }
        if (cudaFuncSetAttribute(p2p_monopole_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, MONO_SMEM) != cudaSuccess) {
            delete h; return OCTO_FMM_ECUDA;
        }
        // ---- tensor-core kernels: tables of A fragments (build_dmma_table) ----
        {
            std::vector<DmmaEntry> tab((size_t)4 * DMMA_MAX_CHUNKS * 32 + (size_t)DMMA_MAX_CHUNKS_POT * 32, DmmaEntry{0.0, 0, 0});
            for (int which = 0; which < 5; ++which) {
                DmmaRow rows[8];
                dmma_rows(h->list, which, rows);
                const int n = build_dmma_table(rows, wt, tab.data() + (size_t)which * DMMA_MAX_CHUNKS * 32,
                                               which < 4 ? DMMA_MAX_CHUNKS : DMMA_MAX_CHUNKS_POT);
                if (n < 0) { delete h; return OCTO_FMM_EINVAL; }
                if (which < 4) h->dl.nchunk[which] = n; else h->nchunk_pot = n;
            }
            if (cudaMemcpyAsync(h->T, tab.data(), tab.size() * sizeof(DmmaEntry), cudaMemcpyHostToDevice, h->stream) != cudaSuccess ||
                cudaStreamSynchronize(h->stream) != cudaSuccess) { delete h; return OCTO_FMM_ECUDA; }
            cuuint32_t mbox2[3] = {MS_XH, 2 * MS_Y, DS_Z};
            std::memset(&h->tmap2, 0, sizeof(h->tmap2));
            if (enc(&h->tmap2, CU_TENSOR_MAP_DATA_TYPE_FLOAT64, 3, (void*)h->src, mdims, mstrides, mbox2, mestr, CU_TENSOR_MAP_INTERLEAVE_NONE,
                    CU_TENSOR_MAP_SWIZZLE_NONE, CU_TENSOR_MAP_L2_PROMOTION_L2_128B, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE) != CUDA_SUCCESS) {
                delete h; return OCTO_FMM_ECUDA;
            }
            if (cudaFuncSetAttribute(p2p_monopole_dmma_kernel<false>, cudaFuncAttributeMaxDynamicSharedMemorySize, DMMA_SMEM) != cudaSuccess ||
                cudaFuncSetAttribute(p2p_monopole_dmma_kernel<true>, cudaFuncAttributeMaxDynamicSharedMemorySize, DMMA_SMEM) != cudaSuccess ||
                cudaFuncSetAttribute(p2p_potential_dmma_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, DMMA_SMEM) != cudaSuccess) {
                delete h; return OCTO_FMM_ECUDA;
            }
        }
    }
    *out = h;
    return OCTO_FMM_OK;
}

int octo_fmm_create(const octo_fmm_config* cfg, octo_fmm_t** out) { return create_internal(cfg, 0, out); }

int octo_fmm_set_moments(octo_fmm_t* h, const double* moments, const double* com_off)
{
    if (!h || !moments) return OCTO_FMM_EINVAL;
    if (cudaSetDevice(h->cfg.device) != cudaSuccess) return OCTO_FMM_ECUDA;
    const Params& P = h->prm;
    if (h->cfg.kind == OCTO_FMM_MULTIPOLE) {
        const long long ncell = (long long)P.nx * P.ny * P.nz;
        if (cudaMemsetAsync(h->flags + 1, 0, sizeof(int), h->stream) != cudaSuccess) return OCTO_FMM_ECUDA;
        stage_multipole_kernel<<<(unsigned)((ncell + 255) / 256), 256, 0, h->stream>>>(moments, com_off, h->src, P.nx, P.ny, P.nz,
                                                                                       0, P.nz, h->cfg.h, h->flags, h->cfg.am_correction);
    } else {
        const long long pc = (long long)(P.nx + REACH_MAX + MONO_PAD_RIGHT) * (P.ny + 2 * REACH_MAX) * (P.nz + 2 * REACH_MAX);
        stage_monopole_kernel<<<(unsigned)((pc + 255) / 256), 256, 0, h->stream>>>(moments, h->src, P.nx, P.ny, P.nz);
    }
    if (cudaGetLastError() != cudaSuccess) return OCTO_FMM_ECUDA;
    h->state = 1;
    return OCTO_FMM_OK;
}

// Make the lists of h current in the device's constant bank for a kernel about to be launched on h->stream, then
// (bank_reader_done) note that kernel as a reader.  The caller holds BankLock from before bank_acquire until after
// bank_reader_done, so that no other host thread can slip an upload between the two.
struct BankLock {
    std::unique_lock<std::mutex> lk;
    explicit BankLock(const octo_fmm_t* h);
};

static int bank_acquire(octo_fmm_t* h, bool mixed = false)
{
    ConstBank& b = g_bank[h->cfg.device];
    const unsigned long long sig = mixed ? h->list_sig_mixed : h->list_sig;
    if (b.sig == sig) {
        // same lists; if they were uploaded on another stream, this stream has to see the upload complete
        if (b.up_stream != h->stream && b.uploaded && cudaStreamWaitEvent(h->stream, b.uploaded, 0) != cudaSuccess) return OCTO_FMM_ECUDA;
        return OCTO_FMM_OK;
    }
    // other lists: wait for every kernel on OTHER streams that still reads the old contents (same-stream readers are
    // ordered before the upload by the stream itself)
    for (auto& r : b.readers) {
        if (r.first != h->stream && cudaStreamWaitEvent(h->stream, r.second, 0) != cudaSuccess) return OCTO_FMM_ECUDA;
        b.pool.push_back(r.second);
    }
    b.readers.clear();
    const StEntry* ent = mixed ? h->entries_mixed.data() : h->entries.data();
    const void* beg = mixed ? (const void*)h->begin_mixed : (const void*)h->begin;
    b.sig = 0;                                        // nothing valid until every piece is on its way
    if (cudaMemcpyToSymbolAsync(c_entries, ent, (size_t)8 * MAX_LIST * sizeof(StEntry), 0, cudaMemcpyHostToDevice, h->stream) != cudaSuccess ||
        cudaMemcpyToSymbolAsync(c_begin, beg, sizeof(h->begin), 0, cudaMemcpyHostToDevice, h->stream) != cudaSuccess ||
        cudaMemcpyToSymbolAsync(c_near, h->near_list.data(), h->near_list.size() * sizeof(char4), 0, cudaMemcpyHostToDevice, h->stream) != cudaSuccess ||
        cudaMemcpyToSymbolAsync(c_near_count, h->near_count, sizeof(h->near_count), 0, cudaMemcpyHostToDevice, h->stream) != cudaSuccess)
        return OCTO_FMM_ECUDA;
    if (!b.uploaded && cudaEventCreateWithFlags(&b.uploaded, cudaEventDisableTiming) != cudaSuccess) return OCTO_FMM_ECUDA;
    if (cudaEventRecord(b.uploaded, h->stream) != cudaSuccess) return OCTO_FMM_ECUDA;
    b.up_stream = h->stream;
    b.sig = sig;
    return OCTO_FMM_OK;
}

static int bank_reader_done(octo_fmm_t* h)
{
    ConstBank& b = g_bank[h->cfg.device];
    for (auto& r : b.readers)
        if (r.first == h->stream) return cudaEventRecord(r.second, h->stream) == cudaSuccess ? OCTO_FMM_OK : OCTO_FMM_ECUDA;
    cudaEvent_t ev = nullptr;
    if (!b.pool.empty()) { ev = b.pool.back(); b.pool.pop_back(); }
    else if (cudaEventCreateWithFlags(&ev, cudaEventDisableTiming) != cudaSuccess) return OCTO_FMM_ECUDA;
    if (cudaEventRecord(ev, h->stream) != cudaSuccess) { b.pool.push_back(ev); return OCTO_FMM_ECUDA; }
    b.readers.emplace_back(h->stream, ev);
    return OCTO_FMM_OK;
}

BankLock::BankLock(const octo_fmm_t* h) : lk(g_bank[h->cfg.device].mu) {}

// true if the kernel interact() launches for this handle reads the constant bank (the tensor-core monopole kernels read
// only their own tables in the workspace)
static bool reads_bank(const octo_fmm_t* h) { return h->cfg.kind == OCTO_FMM_MULTIPOLE || h->mono_kernel != 0; }

// launch the staged interaction kernel for the z-layers [kb, ke) of the output region
static int launch_staged(octo_fmm_t* h, int kb, int ke, bool mixed = false)
{
    Params P = h->prm;
    P.L = h->outL; P.C = h->outC;
    P.kb = kb; P.ke = ke;
    P.tiles_z = (ke - kb + TILE_Z - 1) / TILE_Z;
    P.ntiles = (long long)P.tiles_x * P.tiles_y * P.tiles_z;
    if (h->tile_list) { P.tile_list = h->tile_list; P.tile_zmask = h->tile_zmask; P.ntiles = h->tile_count; }     // whole-grid launches only (tree levels)
    const int grid = (int)std::min<long long>(P.ntiles, h->sm_count);
    if (grid == 0) return OCTO_FMM_OK;
    if (h->tree_kind) {    // a level of the adaptive tree: absent cells, leaf-leaf pairs left to the leaf kernel
        P.leaf = h->tree_kind;
        // one brick per CTA, heaviest first: the levels of a tree run side by side on streams of their own, and the block
        // scheduler packs their bricks onto the SMs as they come free (the ring fill per brick is 3 % of a full brick)
        const int tgrid = (int)P.ntiles;
        if (P.pL) {        // the parent's expansion added in the epilogue (levels one after the other)
            if (h->cfg.am_correction) m2l_staged_kernel<true, true, MODE_TREE><<<tgrid, STAGED_THREADS, STAGED_SMEM, h->stream>>>(h->maps, P);
            else                      m2l_staged_kernel<false, true, MODE_TREE><<<tgrid, STAGED_THREADS, STAGED_SMEM, h->stream>>>(h->maps, P);
        } else {
            if (h->cfg.am_correction) m2l_staged_kernel<true, false, MODE_TREE><<<tgrid, STAGED_THREADS, STAGED_SMEM, h->stream>>>(h->maps, P);
            else                      m2l_staged_kernel<false, false, MODE_TREE><<<tgrid, STAGED_THREADS, STAGED_SMEM, h->stream>>>(h->maps, P);
        }
    } else if (mixed) {    // one level of an adaptive mesh: leaf-level lists, near-field entries conditional on the leaf flags
        if (h->cfg.am_correction) m2l_staged_kernel<true, false, MODE_MIXED><<<grid, STAGED_THREADS, STAGED_SMEM, h->stream>>>(h->maps, P);
        else                      m2l_staged_kernel<false, false, MODE_MIXED><<<grid, STAGED_THREADS, STAGED_SMEM, h->stream>>>(h->maps, P);
    } else if (P.pL) {     // complete solve: L2L fused into the epilogue (solver.inl sets the parent arrays)
        if (h->cfg.am_correction) m2l_staged_kernel<true, true><<<grid, STAGED_THREADS, STAGED_SMEM, h->stream>>>(h->maps, P);
        else                      m2l_staged_kernel<false, true><<<grid, STAGED_THREADS, STAGED_SMEM, h->stream>>>(h->maps, P);
    } else {
        if (h->cfg.am_correction) m2l_staged_kernel<true><<<grid, STAGED_THREADS, STAGED_SMEM, h->stream>>>(h->maps, P);
        else                      m2l_staged_kernel<false><<<grid, STAGED_THREADS, STAGED_SMEM, h->stream>>>(h->maps, P);
    }
    return cudaGetLastError() == cudaSuccess ? OCTO_FMM_OK : OCTO_FMM_ECUDA;
}

static int mono_blocks(const Params& P)
{
    return ((P.ox + MT_X - 1) / MT_X) * ((P.oy + MT_Y - 1) / MT_Y) * ((P.oz + MT_Z - 1) / MT_Z);
}
static int dmma_blocks(const Params& P)
{
    return ((P.ox + MT_X - 1) / MT_X) * ((P.oy + MT_Y - 1) / MT_Y) * ((P.oz + DT_Z - 1) / DT_Z);
}

static int brick_blocks(const Params& P) { return ((P.ox + 15) / 16) * ((P.oy + 7) / 8) * ((P.oz + 3) / 4); }

int octo_fmm_interact(octo_fmm_t* h)
{
    if (!h) return OCTO_FMM_EINVAL;
    if (h->state < 1) return OCTO_FMM_ESTATE;
    if (cudaSetDevice(h->cfg.device) != cudaSuccess) return OCTO_FMM_ECUDA;
    const bool bank = reads_bank(h);
    BankLock guard(h);
    if (!bank) guard.lk.unlock();
    else if (bank_acquire(h) != OCTO_FMM_OK) return OCTO_FMM_ECUDA;
    if (cudaMemsetAsync(h->flags, 0, sizeof(int), h->stream) != cudaSuccess) return OCTO_FMM_ECUDA;
    Params& P = h->prm;
    P.L = h->outL; P.C = h->outC;
    if (h->cfg.kind == OCTO_FMM_MONOPOLE) {
        if (h->tile_list) {                     // a level of the adaptive tree: only the tiles that hold leaves
            if (h->mono_kernel != 0) return OCTO_FMM_ESTATE;
            Params Q = P;
            Q.tile_list = h->tile_list;
            if (h->tile_count > 0)
                p2p_monopole_dmma_kernel<false><<<h->tile_count, DMMA_THREADS, DMMA_SMEM, h->stream>>>(h->tmap2, Q, h->T, h->dl, h->outL);
        } else if (h->mono_kernel == 0) {
            // all tiles, or (host entry points) the z-tiles [mono_zt_begin, mono_zt_end) only
            const int per_z = ((P.ox + MT_X - 1) / MT_X) * ((P.oy + MT_Y - 1) / MT_Y);
            Params Q = P;
            int blocks = dmma_blocks(P);
            if (h->mono_zt_end > 0) { Q.tile_offset = h->mono_zt_begin * per_z; blocks = (h->mono_zt_end - h->mono_zt_begin) * per_z; }
            if (blocks <= 0) return OCTO_FMM_EINVAL;
            if (P.pL)      // complete solve: leaf evaluation fused into the epilogue (solver.inl)
                p2p_monopole_dmma_kernel<true><<<blocks, DMMA_THREADS, DMMA_SMEM, h->stream>>>(h->tmap2, Q, h->T, h->dl, h->outL);
            else
                p2p_monopole_dmma_kernel<false><<<blocks, DMMA_THREADS, DMMA_SMEM, h->stream>>>(h->tmap2, Q, h->T, h->dl, h->outL);
        }
        else
            p2p_monopole_kernel<<<mono_blocks(P), MONO_THREADS, MONO_SMEM, h->stream>>>(h->tmap, P, h->W, h->outL);
    } else if (h->kernel == 1) {
        if (h->cfg.am_correction) m2l_direct_kernel<true><<<brick_blocks(P), 256, 0, h->stream>>>(P);
        else                      m2l_direct_kernel<false><<<brick_blocks(P), 256, 0, h->stream>>>(P);
    } else if (h->kernel == 2) {
        const unsigned blocks = (unsigned)(((long long)P.ox * P.oy * P.oz + 7) / 8);
        if (h->cfg.am_correction) m2l_warp_kernel<true><<<blocks, 256, 0, h->stream>>>(P);
        else                      m2l_warp_kernel<false><<<blocks, 256, 0, h->stream>>>(P);
    } else {
        if (launch_staged(h, h->lo[2], h->hi[2]) != OCTO_FMM_OK) return OCTO_FMM_ECUDA;
    }
    if (cudaGetLastError() != cudaSuccess) return OCTO_FMM_ECUDA;
    if (bank && bank_reader_done(h) != OCTO_FMM_OK) return OCTO_FMM_ECUDA;
    h->state = 2;
    h->mixed = false;
    h->resL = h->outL; h->resC = h->outC;
    return OCTO_FMM_OK;
}

// Two right-hand sides in one pass (solver.inl, octo_fmm_solver_solve2): h1 = the density's handle (sources staged,
// correction as configured), h2 = the handle of d(rho)/dt on the same grid (sources staged with the correction off).
// fused_kind: 2 = one warp per cell (m2l_warp2_kernel), 1 = one thread per cell from global memory (m2l_direct2_kernel).
static int interact2(octo_fmm_t* h1, octo_fmm_t* h2, int fused_kind)
{
    if (!h1 || !h2 || h1->cfg.kind != OCTO_FMM_MULTIPOLE || h2->cfg.kind != OCTO_FMM_MULTIPOLE) return OCTO_FMM_EINVAL;
    if (h1->state < 1 || h2->state < 1) return OCTO_FMM_ESTATE;
    for (int a = 0; a < 3; ++a)
        if (h1->cfg.n[a] != h2->cfg.n[a] || h1->lo[a] != h2->lo[a] || h1->hi[a] != h2->hi[a]) return OCTO_FMM_EINVAL;
    if (h2->cfg.am_correction || h1->stream != h2->stream) return OCTO_FMM_EINVAL;
    if (cudaSetDevice(h1->cfg.device) != cudaSuccess) return OCTO_FMM_ECUDA;
    BankLock guard(h1);
    if (bank_acquire(h1) != OCTO_FMM_OK) return OCTO_FMM_ECUDA;
    if (cudaMemsetAsync(h1->flags, 0, sizeof(int), h1->stream) != cudaSuccess) return OCTO_FMM_ECUDA;
    Params P = h1->prm, Q = h2->prm;
    P.L = h1->outL; P.C = h1->outC; P.pL = nullptr;
    Q.L = h2->outL; Q.C = h2->outC; Q.pL = nullptr;
    if (fused_kind == 2) {
        const unsigned blocks = (unsigned)(((long long)P.ox * P.oy * P.oz + 7) / 8);
        if (h1->cfg.am_correction) m2l_warp2_kernel<true><<<blocks, 256, 0, h1->stream>>>(P, Q);
        else                       m2l_warp2_kernel<false><<<blocks, 256, 0, h1->stream>>>(P, Q);
    } else {
        if (h1->cfg.am_correction) m2l_direct2_kernel<true><<<brick_blocks(P), 256, 0, h1->stream>>>(P, Q);
        else                       m2l_direct2_kernel<false><<<brick_blocks(P), 256, 0, h1->stream>>>(P, Q);
    }
    if (cudaGetLastError() != cudaSuccess) return OCTO_FMM_ECUDA;
    if (bank_reader_done(h1) != OCTO_FMM_OK) return OCTO_FMM_ECUDA;
    for (octo_fmm_t* h : {h1, h2}) {
        h->state = 2;
        h->mixed = false;
        h->resL = h->outL; h->resC = h->outC;
    }
    return OCTO_FMM_OK;
}

// number of near-field pairs with a leaf on either side (for the bit-exact check of the pair set)
__global__ void __launch_bounds__(256) count_near_kernel(const Params p, const unsigned char* __restrict__ leaf,
                                                         unsigned long long* __restrict__ count)
{
    const long long o = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    unsigned long long taken = 0;
    if (o < (long long)p.ox * p.oy * p.oz) {
        const int gx = p.lo[0] + (int)(o % p.ox), gy = p.lo[1] + (int)((o / p.ox) % p.oy), k = p.lo[2] + (int)(o / ((long long)p.ox * p.oy));
        const int cls = (gx & 1) + 2 * (gy & 1) + 4 * (k & 1);
        const long long plane = (long long)p.ny * p.nx;
        const bool leafA = leaf[(long long)k * plane + (long long)gy * p.nx + gx] != 0;
        for (int s = 0; s < c_near_count[cls]; ++s) {
            const char4 e = c_near[cls][s];
            const int sx = gx + e.x, sy = gy + e.y, sz = k + e.z;
            if (sx < 0 || sy < 0 || sz < 0 || sx >= p.nx || sy >= p.ny || sz >= p.nz) continue;
            if (leafA || leaf[(long long)sz * plane + (long long)sy * p.nx + sx] != 0) ++taken;
        }
    }
    for (int d = 16; d > 0; d >>= 1) taken += __shfl_xor_sync(0xffffffffu, taken, d);
    if ((threadIdx.x & 31) == 0 && taken) atomicAdd(count, taken);
}

int octo_fmm_interact_mixed(octo_fmm_t* h, const unsigned char* leaf)
{
    if (!h || !leaf || h->cfg.kind != OCTO_FMM_MULTIPOLE) return OCTO_FMM_EINVAL;
    if (h->state < 1 || h->has_neighbours) return OCTO_FMM_ESTATE;
    if (cudaSetDevice(h->cfg.device) != cudaSuccess) return OCTO_FMM_ECUDA;
    if (h->kernel == 0) {
        // slab-fed kernel: one pass over the leaf-level lists; the partner's leaf flag travels in the padding slot of its record
        BankLock guard(h);
        if (bank_acquire(h, true) != OCTO_FMM_OK) return OCTO_FMM_ECUDA;
        if (cudaMemsetAsync(h->flags, 0, sizeof(int), h->stream) != cudaSuccess) return OCTO_FMM_ECUDA;
        Params& P = h->prm;
        const long long ncell = (long long)P.nx * P.ny * P.nz;
        stage_leaf_flags_kernel<<<(unsigned)((ncell + 255) / 256), 256, 0, h->stream>>>(leaf, h->src, P.nx, P.ny, P.nz);
        if (cudaGetLastError() != cudaSuccess) return OCTO_FMM_ECUDA;
        P.leaf = leaf;
        const int rc = launch_staged(h, h->lo[2], h->hi[2], true);
        P.leaf = nullptr;
        if (rc != OCTO_FMM_OK) return rc;
        if (bank_reader_done(h) != OCTO_FMM_OK) return OCTO_FMM_ECUDA;
        h->state = 2;
        h->resL = h->outL; h->resC = h->outC;
    } else {
        const int rc = octo_fmm_interact(h);                   // the Eq. 15 part, whatever the cells' kind
        if (rc != OCTO_FMM_OK) return rc;
        BankLock guard(h);
        if (bank_acquire(h) != OCTO_FMM_OK) return OCTO_FMM_ECUDA;      // the near-field table travels with the lists
        Params P = h->prm;
        P.L = h->outL; P.C = h->outC;
        // the same dipole decision as the interaction kernels (flags[1] or "dipole_terms"), read on the device
        if (h->cfg.am_correction) m2l_near_kernel<true><<<brick_blocks(P), 256, 0, h->stream>>>(P, leaf, nullptr);
        else                      m2l_near_kernel<false><<<brick_blocks(P), 256, 0, h->stream>>>(P, leaf, nullptr);
        if (cudaGetLastError() != cudaSuccess) return OCTO_FMM_ECUDA;
        if (bank_reader_done(h) != OCTO_FMM_OK) return OCTO_FMM_ECUDA;
    }
    h->mixed = true;
    h->mixed_counted = false;
    if (h->mixed_count) {
        unsigned long long* cnt = reinterpret_cast<unsigned long long*>(h->flags + 2);
        if (cudaMemsetAsync(cnt, 0, sizeof(unsigned long long), h->stream) != cudaSuccess) return OCTO_FMM_ECUDA;
        const Params& P = h->prm;
        const long long ocell = (long long)P.ox * P.oy * P.oz;
        BankLock guard(h);
        if (bank_acquire(h, h->kernel == 0) != OCTO_FMM_OK) return OCTO_FMM_ECUDA;   // c_near is the same in both flavours: no re-upload
        count_near_kernel<<<(unsigned)((ocell + 255) / 256), 256, 0, h->stream>>>(P, leaf, cnt);
        if (cudaGetLastError() != cudaSuccess) return OCTO_FMM_ECUDA;
        if (bank_reader_done(h) != OCTO_FMM_OK) return OCTO_FMM_ECUDA;
        h->mixed_counted = true;
    }
    return OCTO_FMM_OK;
}

int octo_fmm_mixed_interaction_count(octo_fmm_t* h, unsigned long long* n)
{
    if (!h || !n) return OCTO_FMM_EINVAL;
    if (h->state < 2 || !h->mixed || !h->mixed_counted) return OCTO_FMM_ESTATE;
    if (cudaStreamSynchronize(h->stream) != cudaSuccess) return OCTO_FMM_ECUDA;
    unsigned long long near = 0;
    if (cudaMemcpy(&near, h->flags + 2, sizeof near, cudaMemcpyDeviceToHost) != cudaSuccess) return OCTO_FMM_ECUDA;
    *n = h->n_interactions + near;
    return OCTO_FMM_OK;
}

// Monopole handles: the potential row only, out = [oz][oy][ox] (second right-hand side of the complete solve).
static int interact_potential(octo_fmm_t* h, double* out)
{
    if (!h || !out || h->cfg.kind != OCTO_FMM_MONOPOLE) return OCTO_FMM_EINVAL;
    if (h->state < 1) return OCTO_FMM_ESTATE;
    if (cudaSetDevice(h->cfg.device) != cudaSuccess) return OCTO_FMM_ECUDA;
    const Params& P = h->prm;
    p2p_potential_dmma_kernel<<<dmma_blocks(P), DMMA_THREADS, DMMA_SMEM, h->stream>>>(
        h->tmap2, P, h->T + (size_t)4 * DMMA_MAX_CHUNKS * 32, h->nchunk_pot, out);
    return cudaGetLastError() == cudaSuccess ? OCTO_FMM_OK : OCTO_FMM_ECUDA;
}

int octo_fmm_bind_outputs(octo_fmm_t* h, double* L, double* Lcorr)
{
    if (!h) return OCTO_FMM_EINVAL;
    if (!L && Lcorr) return OCTO_FMM_EINVAL;
    if (Lcorr && h->cfg.kind != OCTO_FMM_MULTIPOLE) return OCTO_FMM_EINVAL;
    h->outL = L ? L : h->L;
    h->outC = (L && Lcorr) ? Lcorr : h->C;
    return OCTO_FMM_OK;
}

int octo_fmm_get_expansions(octo_fmm_t* h, double* L, double* Lcorr)
{
    if (!h || !L) return OCTO_FMM_EINVAL;
    if (h->state < 2) return OCTO_FMM_ESTATE;
    const Params& P = h->prm;
    const size_t ocell = (size_t)P.ox * P.oy * P.oz;
    const size_t ncoef = h->cfg.kind == OCTO_FMM_MULTIPOLE ? 20 : 4;
    // results already in place when interact() wrote into bound caller buffers
    if (L != h->resL &&
        cudaMemcpyAsync(L, h->resL, ocell * ncoef * sizeof(double), cudaMemcpyDeviceToDevice, h->stream) != cudaSuccess)
        return OCTO_FMM_ECUDA;
    if (Lcorr) {
        if (h->cfg.kind != OCTO_FMM_MULTIPOLE) return OCTO_FMM_EINVAL;
        if (Lcorr != h->resC &&
            cudaMemcpyAsync(Lcorr, h->resC, ocell * 3 * sizeof(double), cudaMemcpyDeviceToDevice, h->stream) != cudaSuccess)
            return OCTO_FMM_ECUDA;
    }
    return OCTO_FMM_OK;
}

int octo_fmm_status(octo_fmm_t* h)
{
    if (!h) return OCTO_FMM_EINVAL;
    if (cudaStreamSynchronize(h->stream) != cudaSuccess) return OCTO_FMM_ECUDA;
    if (h->state < 2) return OCTO_FMM_OK;
    int f = 0;
    if (cudaMemcpy(&f, h->flags, sizeof(int), cudaMemcpyDeviceToHost) != cudaSuccess) return OCTO_FMM_ECUDA;
    return (f & 1) ? OCTO_FMM_EMASS : OCTO_FMM_OK;
}

int octo_fmm_dipole_terms_used(octo_fmm_t* h, int* used)
{
    if (!h || !used) return OCTO_FMM_EINVAL;
    if (h->cfg.kind != OCTO_FMM_MULTIPOLE) return OCTO_FMM_EINVAL;
    if (h->state < 1) return OCTO_FMM_ESTATE;
    if (cudaStreamSynchronize(h->stream) != cudaSuccess) return OCTO_FMM_ECUDA;
    int f = 0;
    if (cudaMemcpy(&f, h->flags + 1, sizeof(int), cudaMemcpyDeviceToHost) != cudaSuccess) return OCTO_FMM_ECUDA;
    for (const int* nf : {h->prm.nflags[0], h->prm.nflags[1]}) {      // the neighbours' sources count too (f4)
        int g = 0;
        if (nf && cudaMemcpy(&g, nf + 1, sizeof(int), cudaMemcpyDeviceToHost) != cudaSuccess) return OCTO_FMM_ECUDA;
        f |= g;
    }
    *used = (h->prm.force_dipole || (f & 2)) ? 1 : 0;
    return OCTO_FMM_OK;
}

int octo_fmm_destroy(octo_fmm_t* h)
{
    if (!h) return OCTO_FMM_EINVAL;
    cudaError_t e = cudaStreamSynchronize(h->stream);
    if (h->s_h2d) cudaStreamDestroy(h->s_h2d);
    if (h->s_d2h) cudaStreamDestroy(h->s_d2h);
    for (int i = 0; i < MAX_CHUNKS; ++i) {
        if (h->ev_in[i]) cudaEventDestroy(h->ev_in[i]);
        if (h->ev_out[i]) cudaEventDestroy(h->ev_out[i]);
    }
    if (h->ev_begin) cudaEventDestroy(h->ev_begin);
    if (h->ev_end) cudaEventDestroy(h->ev_end);
    if (h->pinned_flag) cudaFreeHost(h->pinned_flag);
    delete h;
    return e == cudaSuccess ? OCTO_FMM_OK : OCTO_FMM_ECUDA;
}

int octo_fmm_get_stencil(const octo_fmm_t* h, int parity, int* count, signed char (*dxyz)[3])
{
    if (!h || !count || parity < 0 || parity > 7) return OCTO_FMM_EINVAL;
    *count = (int)h->list[parity].size();
    if (dxyz)
        for (size_t s = 0; s < h->list[parity].size(); ++s)
            for (int a = 0; a < 3; ++a) dxyz[s][a] = h->list[parity][s].d[a];
    return OCTO_FMM_OK;
}

int octo_fmm_dmma_table(double theta, double h, int leaf, int which, int cap_chunks, int* nchunk, double* a, int* off)
{
    if (!(theta > 1.0 / 3.0 && theta < 1.0) || !(h > 0.0) || which < 0 || which > 4 || !nchunk || cap_chunks < 0) return OCTO_FMM_EINVAL;
    std::vector<Offset3> list[8];
    int reach = 0;
    for (int p = 0; p < 8; ++p) list[p] = build_list(p & 1, (p >> 1) & 1, (p >> 2) & 1, theta, &reach, leaf != 0);
    if (reach > REACH_MAX) return OCTO_FMM_EINVAL;
    double hmul[2 * REACH_MAX + 1];
    for (int d = -REACH_MAX; d <= REACH_MAX; ++d) hmul[d + REACH_MAX] = (double)(-d) * h;
    const std::vector<double4> wt = monopole_weights(hmul);
    DmmaRow rows[8];
    dmma_rows(list, which, rows);
    const int maxc = which < 4 ? DMMA_MAX_CHUNKS : DMMA_MAX_CHUNKS_POT;
    std::vector<DmmaEntry> tab((size_t)maxc * 32, DmmaEntry{0.0, 0, 0});
    const int n = build_dmma_table(rows, wt, tab.data(), maxc);
    if (n < 0) return OCTO_FMM_EINVAL;
    *nchunk = n;
    if (a && off) {
        if (cap_chunks < n) return OCTO_FMM_EINVAL;
        for (size_t i = 0; i < (size_t)n * 32; ++i) { a[i] = tab[i].a; off[i] = tab[i].off; }
    }
    return OCTO_FMM_OK;
}

int octo_fmm_interaction_count(const octo_fmm_t* h, unsigned long long* n)
{
    if (!h || !n) return OCTO_FMM_EINVAL;
    *n = h->n_interactions;
    return OCTO_FMM_OK;
}

// ---- f4: z-slab sharding with the halo read from peer memory ----
int octo_fmm_staged_sources(const octo_fmm_t* h, octo_fmm_peer* self)
{
    if (!h || !self || h->cfg.kind != OCTO_FMM_MULTIPOLE) return OCTO_FMM_EINVAL;
    self->sources = h->src;
    self->flags = h->flags;
    self->nz = h->cfg.n[2];
    return OCTO_FMM_OK;
}

int octo_fmm_set_neighbours(octo_fmm_t* h, const octo_fmm_peer* below, const octo_fmm_peer* above)
{
    if (!h || h->cfg.kind != OCTO_FMM_MULTIPOLE) return OCTO_FMM_EINVAL;
    // the slab-fed kernel over the whole x-y plane of a plain uniform level only
    if (h->kernel != 0 || h->tree_kind || h->tile_list) return OCTO_FMM_EINVAL;
    for (const octo_fmm_peer* nb : {below, above})
        if (nb && (!nb->sources || !nb->flags || nb->nz < h->reach || ((uintptr_t)nb->sources % 16))) return OCTO_FMM_EINVAL;
    if (cudaSetDevice(h->cfg.device) != cudaSuccess) return OCTO_FMM_ECUDA;
    SlabMaps m = h->maps;
    m.below = m.own; m.above = m.own;
    if (below && encode_slab_map(&m.below, below->sources, h->cfg.n[0], h->cfg.n[1], below->nz) != OCTO_FMM_OK) return OCTO_FMM_ECUDA;
    if (above && encode_slab_map(&m.above, above->sources, h->cfg.n[0], h->cfg.n[1], above->nz) != OCTO_FMM_OK) return OCTO_FMM_ECUDA;
    h->maps = m;
    Params& P = h->prm;
    // only the layers within the stencil's reach are ever read
    P.zmin = below ? -h->reach : 0;
    P.zmax = h->cfg.n[2] - 1 + (above ? h->reach : 0);
    P.nz_below = below ? below->nz : 0;
    P.nflags[0] = below ? below->flags : nullptr;
    P.nflags[1] = above ? above->flags : nullptr;
    h->has_neighbours = below || above;
    h->n_interactions = count_interactions(h, P.zmin, P.zmax);
    return OCTO_FMM_OK;
}

int octo_fmm_ipc_export(const void* dev_ptr, unsigned char handle[64], unsigned long long* offset)
{
    if (!dev_ptr || !handle || !offset) return OCTO_FMM_EINVAL;
    static_assert(sizeof(cudaIpcMemHandle_t) == 64, "CUDA IPC handles are 64 bytes");
    CUdeviceptr base = 0;
    size_t size = 0;
    typedef CUresult (*RangeFn)(CUdeviceptr*, size_t*, CUdeviceptr);
    void* fn = nullptr;
    cudaDriverEntryPointQueryResult q;
    if (cudaGetDriverEntryPoint("cuMemGetAddressRange", &fn, cudaEnableDefault, &q) != cudaSuccess || !fn) return OCTO_FMM_ECUDA;
    if (((RangeFn)fn)(&base, &size, (CUdeviceptr)(uintptr_t)dev_ptr) != CUDA_SUCCESS) return OCTO_FMM_ECUDA;
    cudaIpcMemHandle_t hd;
    if (cudaIpcGetMemHandle(&hd, (void*)(uintptr_t)base) != cudaSuccess) { cudaGetLastError(); return OCTO_FMM_ECUDA; }
    std::memcpy(handle, &hd, 64);
    *offset = (unsigned long long)((uintptr_t)dev_ptr - (uintptr_t)base);
    return OCTO_FMM_OK;
}

int octo_fmm_ipc_import(const unsigned char handle[64], unsigned long long offset, void** base, void** dev_ptr)
{
    if (!handle || !base || !dev_ptr) return OCTO_FMM_EINVAL;
    cudaIpcMemHandle_t hd;
    std::memcpy(&hd, handle, 64);
    void* b = nullptr;
    if (cudaIpcOpenMemHandle(&b, hd, cudaIpcMemLazyEnablePeerAccess) != cudaSuccess) { cudaGetLastError(); return OCTO_FMM_ECUDA; }
    *base = b;
    *dev_ptr = (char*)b + offset;
    return OCTO_FMM_OK;
}

int octo_fmm_ipc_close(void* base)
{
    if (!base) return OCTO_FMM_EINVAL;
    if (cudaIpcCloseMemHandle(base) != cudaSuccess) { cudaGetLastError(); return OCTO_FMM_ECUDA; }
    return OCTO_FMM_OK;
}

// side streams and events of the host entry points, created piece by piece; whatever exists is destroyed by
// octo_fmm_destroy (the handle is zero-initialised)
static int ensure_pipeline(octo_fmm_t* h)
{
    if (h->pipeline_ready) return OCTO_FMM_OK;
    if (!h->s_h2d && cudaStreamCreateWithFlags(&h->s_h2d, cudaStreamNonBlocking) != cudaSuccess) return OCTO_FMM_ECUDA;
    if (!h->s_d2h && cudaStreamCreateWithFlags(&h->s_d2h, cudaStreamNonBlocking) != cudaSuccess) return OCTO_FMM_ECUDA;
    for (int i = 0; i < MAX_CHUNKS; ++i)
        if ((!h->ev_in[i] && cudaEventCreateWithFlags(&h->ev_in[i], cudaEventDisableTiming) != cudaSuccess) ||
            (!h->ev_out[i] && cudaEventCreateWithFlags(&h->ev_out[i], cudaEventDisableTiming) != cudaSuccess)) return OCTO_FMM_ECUDA;
    if ((!h->ev_begin && cudaEventCreateWithFlags(&h->ev_begin, cudaEventDisableTiming) != cudaSuccess) ||
        (!h->ev_end && cudaEventCreateWithFlags(&h->ev_end, cudaEventDisableTiming) != cudaSuccess)) return OCTO_FMM_ECUDA;
    if (!h->pinned_flag && cudaHostAlloc((void**)&h->pinned_flag, 2 * sizeof(int), cudaHostAllocDefault) != cudaSuccess) return OCTO_FMM_ECUDA;
    h->pipeline_ready = true;
    return OCTO_FMM_OK;
}

// Whole step on host buffers, pipelined over slabs of z-layers (multipole kind, staged kernel):
// the host->device copy of slab c+1, the staging + interaction kernels of slab c and the
// device->host copy of slab c-1 run concurrently on three streams (PCIe is full duplex), so the
// step costs about max(H2D, compute, D2H) instead of their sum.  Slab c's output layers
// [a, b) need source layers [a - reach, b + reach): H2D(c) brings every layer of that range that
// earlier slabs have not brought.  Every layer crosses PCIe exactly once in each direction.
static int run_host_pipelined(octo_fmm_t* h, const double* mom_h, const double* com_h, double* L_h, double* C_h,
                              double* d_m, double* d_c, double* d_L, double* d_C)
{
    const Params& P = h->prm;
    if (ensure_pipeline(h) != OCTO_FMM_OK) return OCTO_FMM_ECUDA;
    int zc = h->host_chunk;
    while ((P.oz + zc - 1) / zc + 4 > MAX_CHUNKS) zc += TILE_Z;
    // Slab boundaries.  The bus is the bottleneck, so what the pipeline adds to the pure copy time is its fill (the
    // input of the first slab + halo before the first launch) and its drain (the last launch and its copy out): the
    // first and the last two slabs are short (3 and 6 layers), the others zc.
    int bound[MAX_CHUNKS + 1];
    int nchunk = 0;
    {
        int z = P.lo[2];
        bound[0] = z;
        const bool ramp = P.oz >= 4 * zc && zc > 2 * TILE_Z;
        auto push = [&](int len) { z = std::min(z + len, P.hi[2]); bound[++nchunk] = z; };
        if (ramp) { push(TILE_Z); push(2 * TILE_Z); }
        const int tail = ramp ? 3 * TILE_Z : 0;
        while (P.hi[2] - z > tail + zc) push(zc);
        if (P.hi[2] - z > tail) push(P.hi[2] - z - tail);
        if (ramp) { push(2 * TILE_Z); push(TILE_Z); }
    }
    const size_t plane = (size_t)P.nx * P.ny, ncell = plane * P.nz;
    const size_t oplane = (size_t)P.ox * P.oy, ocell = oplane * P.oz;
    cudaStream_t sm = h->stream;
    BankLock guard(h);                                     // held over all launches of this step
    // interact() is redirected into the caller's scratch for the duration of this call only: restored on EVERY exit
    struct Redirect {
        octo_fmm_t* h; double* L; double* C;
        Redirect(octo_fmm_t* h_, double* nl, double* nc) : h(h_), L(h_->outL), C(h_->outC) { h->outL = nl; h->outC = nc; }
        ~Redirect() { h->outL = L; h->outC = C; }
    } redirect(h, d_L, d_C);
#define OCTO_TRY(call) do { if ((call) != cudaSuccess) return OCTO_FMM_ECUDA; } while (0)
    auto body = [&]() -> int {
    OCTO_TRY(cudaMemsetAsync(h->flags, 0, 2 * sizeof(int), sm));
    if (bank_acquire(h) != OCTO_FMM_OK) return OCTO_FMM_ECUDA;
    OCTO_TRY(cudaEventRecord(h->ev_begin, sm));            // the copies start after earlier work on the caller's stream
    OCTO_TRY(cudaStreamWaitEvent(h->s_h2d, h->ev_begin, 0));
    OCTO_TRY(cudaStreamWaitEvent(h->s_d2h, h->ev_begin, 0));
    int brought = std::max(P.lo[2] - h->reach, 0);         // source layers [.., brought) are on the device
    int rc = OCTO_FMM_OK;
    for (int c = 0; c < nchunk && rc == OCTO_FMM_OK; ++c) {
        const int a = bound[c], b = bound[c + 1];
        const int need = std::min(b + h->reach, P.nz);
        if (need > brought) {
            const size_t off = (size_t)brought * plane, width = (size_t)(need - brought) * plane * 8;
            OCTO_TRY(cudaMemcpy2DAsync(d_m + off, ncell * 8, mom_h + off, ncell * 8, width, 20, cudaMemcpyHostToDevice, h->s_h2d));
            OCTO_TRY(cudaMemcpy2DAsync(d_c + off, ncell * 8, com_h + off, ncell * 8, width, 3, cudaMemcpyHostToDevice, h->s_h2d));
        }
        OCTO_TRY(cudaEventRecord(h->ev_in[c], h->s_h2d));
        OCTO_TRY(cudaStreamWaitEvent(sm, h->ev_in[c], 0));
        if (need > brought) {
            const long long n = (long long)(need - brought) * (long long)plane;
            stage_multipole_kernel<<<(unsigned)((n + 255) / 256), 256, 0, sm>>>(d_m, d_c, h->src, P.nx, P.ny, P.nz, brought,
                                                                                 need - brought, h->cfg.h, h->flags, h->cfg.am_correction);
            OCTO_TRY(cudaGetLastError());
            brought = need;
        }
        rc = launch_staged(h, a, b);
        if (rc != OCTO_FMM_OK) break;
        OCTO_TRY(cudaEventRecord(h->ev_out[c], sm));
        OCTO_TRY(cudaStreamWaitEvent(h->s_d2h, h->ev_out[c], 0));
        const size_t ooff = (size_t)(a - P.lo[2]) * oplane, owidth = (size_t)(b - a) * oplane * 8;
        OCTO_TRY(cudaMemcpy2DAsync(L_h + ooff, ocell * 8, d_L + ooff, ocell * 8, owidth, 20, cudaMemcpyDeviceToHost, h->s_d2h));
        if (C_h)
            OCTO_TRY(cudaMemcpy2DAsync(C_h + ooff, ocell * 8, d_C + ooff, ocell * 8, owidth, 3, cudaMemcpyDeviceToHost, h->s_d2h));
    }
    if (rc != OCTO_FMM_OK) return rc;
    if (bank_reader_done(h) != OCTO_FMM_OK) return OCTO_FMM_ECUDA;
    OCTO_TRY(cudaEventRecord(h->ev_end, h->s_d2h));
    OCTO_TRY(cudaStreamWaitEvent(sm, h->ev_end, 0));        // the caller's stream completes when the last copy has
    return OCTO_FMM_OK;
    };
#undef OCTO_TRY
    const int rc = body();
    if (rc != OCTO_FMM_OK) {
        // join the side streams so that nothing of this call is still in flight when the caller frees its buffers
        cudaStreamSynchronize(h->s_h2d);
        cudaStreamSynchronize(h->s_d2h);
        return rc;
    }
    h->host_launches = 2 * nchunk;
    return OCTO_FMM_OK;
}

int octo_fmm_run_host(octo_fmm_t* h, const double* moments_host, const double* com_off_host, double* L_host,
                      double* Lcorr_host, void* scratch, size_t scratch_bytes)
{
    if (!h || !moments_host || !L_host || !scratch) return OCTO_FMM_EINVAL;
    if (h->has_neighbours) return OCTO_FMM_ESTATE;     // the neighbours' staging is ordered by the caller, not by this call
    if (scratch_bytes < octo_fmm_host_scratch_bytes(&h->cfg) || ((uintptr_t)scratch % ALIGN)) return OCTO_FMM_EINVAL;
    const Params& P = h->prm;
    const size_t ncell = (size_t)P.nx * P.ny * P.nz, ocell = (size_t)P.ox * P.oy * P.oz;
    const bool multi = h->cfg.kind == OCTO_FMM_MULTIPOLE;
    if (multi && !com_off_host) return OCTO_FMM_EINVAL;
    if (!multi && Lcorr_host) return OCTO_FMM_EINVAL;
    char* w = (char*)scratch;
    double* d_m = (double*)w; w += align_up(ncell * (multi ? 20 : 1) * 8);
    double* d_c = nullptr;
    if (multi) { d_c = (double*)w; w += align_up(ncell * 3 * 8); }
    double* d_L = (double*)w; w += align_up(ocell * (multi ? 20 : 4) * 8);
    double* d_C = multi ? (double*)w : nullptr;
    if (cudaSetDevice(h->cfg.device) != cudaSuccess) return OCTO_FMM_ECUDA;
    if (ensure_pipeline(h) != OCTO_FMM_OK) return OCTO_FMM_ECUDA;
    if (multi && h->kernel == 0 && h->host_chunk > 0) {
        const int rc = run_host_pipelined(h, moments_host, com_off_host, L_host, Lcorr_host, d_m, d_c, d_L, d_C);
        if (rc != OCTO_FMM_OK) return rc;
    } else if (!multi && h->mono_kernel == 0 && !h->tile_list && h->host_chunk > 0) {
        // monopole kind on the tensor-core kernel: the level is launched in chunks of z-tiles and every chunk of the
        // result goes back on a side stream while the next chunks are computed (the outputs are 4x the inputs)
        if (cudaMemcpyAsync(d_m, moments_host, ncell * 8, cudaMemcpyHostToDevice, h->stream) != cudaSuccess) return OCTO_FMM_ECUDA;
        int rc = octo_fmm_set_moments(h, d_m, nullptr);
        if (rc != OCTO_FMM_OK) return rc;
        double* const keepL = h->outL;
        h->outL = d_L;
        const int ztiles = (P.oz + DT_Z - 1) / DT_Z, nchunk = std::min(8, ztiles);
        const size_t oplane = (size_t)P.ox * P.oy;
        for (int c = 0; c < nchunk && rc == OCTO_FMM_OK; ++c) {
            const int a = (int)((long long)ztiles * c / nchunk), b = (int)((long long)ztiles * (c + 1) / nchunk);
            h->mono_zt_begin = a; h->mono_zt_end = b;
            rc = octo_fmm_interact(h);
            if (rc != OCTO_FMM_OK) break;
            const int z0 = a * DT_Z, z1 = std::min(b * DT_Z, P.oz);
            if (cudaEventRecord(h->ev_out[c], h->stream) != cudaSuccess || cudaStreamWaitEvent(h->s_d2h, h->ev_out[c], 0) != cudaSuccess ||
                cudaMemcpy2DAsync(L_host + (size_t)z0 * oplane, ocell * 8, d_L + (size_t)z0 * oplane, ocell * 8,
                                  (size_t)(z1 - z0) * oplane * 8, 4, cudaMemcpyDeviceToHost, h->s_d2h) != cudaSuccess)
                rc = OCTO_FMM_ECUDA;
        }
        h->mono_zt_begin = 0; h->mono_zt_end = 0;
        h->outL = keepL;
        if (rc == OCTO_FMM_OK && (cudaEventRecord(h->ev_end, h->s_d2h) != cudaSuccess || cudaStreamWaitEvent(h->stream, h->ev_end, 0) != cudaSuccess))
            rc = OCTO_FMM_ECUDA;
        if (rc != OCTO_FMM_OK) { cudaStreamSynchronize(h->s_d2h); return rc; }
    } else {
        if (cudaMemcpyAsync(d_m, moments_host, ncell * (multi ? 20 : 1) * 8, cudaMemcpyHostToDevice, h->stream) != cudaSuccess)
            return OCTO_FMM_ECUDA;
        if (multi && cudaMemcpyAsync(d_c, com_off_host, ncell * 3 * 8, cudaMemcpyHostToDevice, h->stream) != cudaSuccess)
            return OCTO_FMM_ECUDA;
        int rc;
        double* const keepL = h->outL; double* const keepC = h->outC;
        if ((rc = octo_fmm_set_moments(h, d_m, d_c)) != OCTO_FMM_OK) return rc;
        h->outL = d_L; h->outC = multi ? d_C : nullptr;       // interact() writes straight into the scratch
        rc = octo_fmm_interact(h);
        h->outL = keepL; h->outC = keepC;
        if (rc != OCTO_FMM_OK) return rc;
        if (cudaMemcpyAsync(L_host, d_L, ocell * (multi ? 20 : 4) * 8, cudaMemcpyDeviceToHost, h->stream) != cudaSuccess)
            return OCTO_FMM_ECUDA;
        if (Lcorr_host && cudaMemcpyAsync(Lcorr_host, d_C, ocell * 3 * 8, cudaMemcpyDeviceToHost, h->stream) != cudaSuccess)
            return OCTO_FMM_ECUDA;
    }
    // the device flag word rides home behind the results, into pinned memory: one synchronisation, no pageable copy
    if (cudaMemcpyAsync(h->pinned_flag, h->flags, sizeof(int), cudaMemcpyDeviceToHost, h->stream) != cudaSuccess) return OCTO_FMM_ECUDA;
    if (cudaStreamSynchronize(h->stream) != cudaSuccess) return OCTO_FMM_ECUDA;
    h->state = 1;                       // the results went to the host; nothing is kept in the scratch
    h->resL = h->L; h->resC = h->C;
    return (h->pinned_flag[0] & 1) ? OCTO_FMM_EMASS : OCTO_FMM_OK;
}

int octo_fmm_set_option(octo_fmm_t* h, const char* key, int value)
{
    if (!h || !key) return OCTO_FMM_EINVAL;
    if (!std::strcmp(key, "kernel")) {
        if (value != 0 && value != 1 && value != 2) return OCTO_FMM_EINVAL;
        if (value == 0 && (h->cfg.n[0] % 8 || h->cfg.n[1] % 8 || h->cfg.n[2] % 8)) return OCTO_FMM_EINVAL;
        h->kernel = value;
        return OCTO_FMM_OK;
    }
    if (!std::strcmp(key, "mono_kernel")) {      // monopole handles: 0 = FP64 tensor-core instruction (default), 1 = DFMA
        if (h->cfg.kind != OCTO_FMM_MONOPOLE || (value != 0 && value != 1)) return OCTO_FMM_EINVAL;
        h->mono_kernel = value;
        return OCTO_FMM_OK;
    }
    if (!std::strcmp(key, "mixed_count")) {      // 1: octo_fmm_interact_mixed also counts the pairs it evaluates
        if (value != 0 && value != 1) return OCTO_FMM_EINVAL;
        h->mixed_count = value;
        return OCTO_FMM_OK;
    }
    if (!std::strcmp(key, "am_correction")) {    // multipole handles: switch the correction for the next set_moments() + interact()
        if (h->cfg.kind != OCTO_FMM_MULTIPOLE || (value != 0 && value != 1)) return OCTO_FMM_EINVAL;
        h->cfg.am_correction = value;
        h->state = 0;                            // the staged sources depend on it: set_moments() again
        return OCTO_FMM_OK;
    }
    if (!std::strcmp(key, "dipole_terms")) {     // 0 = decided on the device from the staged sources (default), 1 = always
        if (value != 0 && value != 1) return OCTO_FMM_EINVAL;
        h->prm.force_dipole = value;
        return OCTO_FMM_OK;
    }
    if (!std::strcmp(key, "host_chunk")) {       // z-layers per run_host pipeline slab; 0 = one copy, one launch
        if (value < 0 || value > 4096) return OCTO_FMM_EINVAL;
        h->host_chunk = value;
        return OCTO_FMM_OK;
    }
    return OCTO_FMM_EINVAL;
}

int octo_fmm_launch_info(const octo_fmm_t* h, int* grid, int* block, int* smem_bytes, int* regs, int* launches)
{
    if (!h) return OCTO_FMM_EINVAL;
    const Params& P = h->prm;
    cudaFuncAttributes fa;
    cudaError_t e;
    int g, b, s;
    if (h->cfg.kind == OCTO_FMM_MONOPOLE && h->mono_kernel == 0) {
        e = cudaFuncGetAttributes(&fa, p2p_monopole_dmma_kernel<false>);
        g = dmma_blocks(P); b = DMMA_THREADS; s = DMMA_SMEM;
    } else if (h->cfg.kind == OCTO_FMM_MONOPOLE) {
        e = cudaFuncGetAttributes(&fa, p2p_monopole_kernel);
        g = mono_blocks(P); b = MONO_THREADS; s = MONO_SMEM;
    } else if (h->kernel == 1) {
        e = h->cfg.am_correction ? cudaFuncGetAttributes(&fa, m2l_direct_kernel<true>) : cudaFuncGetAttributes(&fa, m2l_direct_kernel<false>);
        g = brick_blocks(P); b = 256; s = 0;
    } else if (h->kernel == 2) {
        e = h->cfg.am_correction ? cudaFuncGetAttributes(&fa, m2l_warp_kernel<true>) : cudaFuncGetAttributes(&fa, m2l_warp_kernel<false>);
        g = (int)(((long long)P.ox * P.oy * P.oz + 7) / 8); b = 256; s = 0;
    } else {
        e = h->cfg.am_correction ? cudaFuncGetAttributes(&fa, m2l_staged_kernel<true>) : cudaFuncGetAttributes(&fa, m2l_staged_kernel<false>);
        g = (int)std::min<long long>(P.ntiles, h->sm_count); b = STAGED_THREADS; s = STAGED_SMEM;
    }
    if (e != cudaSuccess) return OCTO_FMM_ECUDA;
    if (grid) *grid = g;
    if (block) *block = b;
    if (smem_bytes) *smem_bytes = s;
    if (regs) *regs = fa.numRegs;
    if (launches) *launches = 1;
    return OCTO_FMM_OK;
}

int octo_fmm_fp64_peak_probe(int device, void* stream, void* scratch, int iters, double* flops_per_s, int* sm_count,
                             int* clock_khz)
{
    if (!scratch || iters <= 0 || !flops_per_s) return OCTO_FMM_EINVAL;
    if (cudaSetDevice(device) != cudaSuccess) return OCTO_FMM_ECUDA;
    cudaDeviceProp prop;
    if (cudaGetDeviceProperties(&prop, device) != cudaSuccess) return OCTO_FMM_ECUDA;
    cudaStream_t st = (cudaStream_t)stream;
    const int blocks = prop.multiProcessorCount * 8;   // 8 x 256 threads = 2048 threads per SM
    if ((size_t)blocks * 256 * 8 > (size_t)8 * 1024 * 1024) return OCTO_FMM_EINVAL;
    cudaEvent_t e0, e1;
    if (cudaEventCreate(&e0) != cudaSuccess || cudaEventCreate(&e1) != cudaSuccess) return OCTO_FMM_ECUDA;
    dfma_peak_kernel<<<blocks, 256, 0, st>>>((double*)scratch, iters / 8 + 1, 1.0);   // warm-up
    cudaEventRecord(e0, st);
    dfma_peak_kernel<<<blocks, 256, 0, st>>>((double*)scratch, iters, 1.0);
    cudaEventRecord(e1, st);
    cudaError_t e = cudaEventSynchronize(e1);
    float ms = 0.f;
    cudaEventElapsedTime(&ms, e0, e1);
    cudaEventDestroy(e0);
    cudaEventDestroy(e1);
    if (e != cudaSuccess || cudaGetLastError() != cudaSuccess) return OCTO_FMM_ECUDA;
    *flops_per_s = (double)blocks * 256.0 * (double)iters * 64.0 * 2.0 / (ms * 1e-3);
    if (sm_count) *sm_count = prop.multiProcessorCount;
    if (clock_khz) *clock_khz = prop.clockRate;
    return OCTO_FMM_OK;
}

int octo_fmm_fp64_issue_probe(int device, void* stream, void* scratch, int mode, int iters, double* instr_per_s)
{
    if (!scratch || iters <= 0 || !instr_per_s || mode < 0 || mode > 2) return OCTO_FMM_EINVAL;
    if (cudaSetDevice(device) != cudaSuccess) return OCTO_FMM_ECUDA;
    cudaDeviceProp prop;
    if (cudaGetDeviceProperties(&prop, device) != cudaSuccess) return OCTO_FMM_ECUDA;
    cudaStream_t st = (cudaStream_t)stream;
    const int blocks = prop.multiProcessorCount, threads = 384;     // 12 warps per SM, as the interaction kernel
    double* out = (double*)scratch;
    double* in = out + (size_t)blocks * threads;
    if (((size_t)blocks * threads + 1024) * 8 > (size_t)8 * 1024 * 1024) return OCTO_FMM_EINVAL;
    if (cudaMemsetAsync(in, 0, 1024 * 8, st) != cudaSuccess) return OCTO_FMM_ECUDA;
    cudaEvent_t e0, e1;
    if (cudaEventCreate(&e0) != cudaSuccess || cudaEventCreate(&e1) != cudaSuccess) return OCTO_FMM_ECUDA;
    for (int pass = 0; pass < 2; ++pass) {
        const int n = pass ? iters : iters / 8 + 1;
        if (pass) cudaEventRecord(e0, st);
        if (mode == 0) fp64_issue_probe_kernel<0><<<blocks, threads, 0, st>>>(out, in, n);
        else if (mode == 1) fp64_issue_probe_kernel<1><<<blocks, threads, 0, st>>>(out, in, n);
        else fp64_issue_probe_kernel<2><<<blocks, threads, 0, st>>>(out, in, n);
    }
    cudaEventRecord(e1, st);
    cudaError_t e = cudaEventSynchronize(e1);
    float ms = 0.f;
    cudaEventElapsedTime(&ms, e0, e1);
    cudaEventDestroy(e0);
    cudaEventDestroy(e1);
    if (e != cudaSuccess || cudaGetLastError() != cudaSuccess) return OCTO_FMM_ECUDA;
    *instr_per_s = (double)blocks * threads * (double)iters * 64.0 / (ms * 1e-3);   // thread-level FP64 instructions
    return OCTO_FMM_OK;
}

int octo_fmm_flops_per_interaction_path(int kind, int am_correction, int dipole_terms, int* flops, int* fp64_instructions)
{
    // What the hot loops of THIS library execute per pair, counted in their SASS (python -m
    // paper_2101_08226_b200.sass_cost_model): DFMA = 2 flop, DADD/DMUL = 1.
    int f, i;
    if (kind == OCTO_FMM_MONOPOLE) { f = 8; i = 4; }
    else if (kind == OCTO_FMM_MULTIPOLE) {
        if (am_correction) {
            if (dipole_terms) { f = 212; i = 130; }   // 82 DFMA + 35 DMUL + 13 DADD   (round 1: 86 + 38 + 14 = 224 flop)
            else              { f = 180; i = 113; }   // 67 DFMA + 33 DMUL + 13 DADD   (round 1: 70 + 34 + 14 = 188 flop)
        } else {
            if (dipole_terms) { f = 202; i = 118; }   // 84 DFMA + 26 DMUL +  8 DADD
            else              { f = 146; i = 90; }    // 56 DFMA + 26 DMUL +  8 DADD
        }
    } else return OCTO_FMM_EINVAL;
    if (flops) *flops = f;
    if (fp64_instructions) *fp64_instructions = i;
    return OCTO_FMM_OK;
}

int octo_fmm_flops_per_interaction(int kind, int am_correction, int* flops, int* fp64_instructions)
{
    return octo_fmm_flops_per_interaction_path(kind, am_correction, 1, flops, fp64_instructions);
}

// ---- the entry point that allocates nothing (octo_fmm.h: octo_fmm_interact_static) ----
// Its scratch -- the staged sources, the flag words, and the result slots a handle's workspace has -- lives in ONE
// file-scope device array: every GPU that loads the library holds these bytes until the process exits.  In host code
// the NAME of the array is a host-side stand-in, not a device address; the address is taken once per device, with that
// device current, by cudaGetSymbolAddress (below) and only that pointer is handed to kernels and to the tensor map.
constexpr size_t STATIC_SCRATCH_BYTES =
    ((size_t)OCTO_FMM_STATIC_MAX_CELLS * (NPAIR * 2 + 20 + 3) * sizeof(double) + 4 * ALIGN + ALIGN - 1) / ALIGN * ALIGN;
static __device__ __align__(256) unsigned char g_static_scratch[STATIC_SCRATCH_BYTES];

struct StaticPath {
    void* scratch = nullptr;       // device address of g_static_scratch on this device
    octo_fmm* h = nullptr;         // handle over the scratch for the configuration of the last call (host memory only)
    octo_fmm_config key{};
};
static StaticPath g_static[MAX_DEVICES];
static std::mutex g_static_mu;

static bool same_static_config(const octo_fmm_config& a, const octo_fmm_config& b)
{
    for (int c = 0; c < 3; ++c)
        if (a.n[c] != b.n[c] || a.out_lo[c] != b.out_lo[c] || a.out_hi[c] != b.out_hi[c]) return false;
    return a.h == b.h && a.theta == b.theta && a.kind == b.kind && a.am_correction == b.am_correction && a.device == b.device &&
           a.stream == b.stream;
}

int octo_fmm_static_max_cells(void) { return OCTO_FMM_STATIC_MAX_CELLS; }

int octo_fmm_interact_static(const octo_fmm_config* cfg, const double* moments, const double* com_off, double* L, double* Lcorr)
{
    if (!cfg || !moments || !L || cfg->kind != OCTO_FMM_MULTIPOLE || !config_ok(cfg)) return OCTO_FMM_EINVAL;
    const long long ncell = (long long)cfg->n[0] * cfg->n[1] * cfg->n[2];
    if (ncell > OCTO_FMM_STATIC_MAX_CELLS) return OCTO_FMM_ESIZE;
    octo_fmm_config c = *cfg;
    c.workspace = nullptr; c.workspace_bytes = 0;
    if (sizes_of(c).total > STATIC_SCRATCH_BYTES) return OCTO_FMM_ESIZE;
    int ndev = 0;
    if (cudaGetDeviceCount(&ndev) != cudaSuccess || c.device < 0 || c.device >= ndev || c.device >= MAX_DEVICES) return OCTO_FMM_ECUDA;
    if (cudaSetDevice(c.device) != cudaSuccess) return OCTO_FMM_ECUDA;
    std::lock_guard<std::mutex> guard(g_static_mu);
    StaticPath& sp = g_static[c.device];
    if (!sp.scratch) {         // set-up, once per device, with that device current
        void* ptr = nullptr;
        if (cudaGetSymbolAddress(&ptr, g_static_scratch) != cudaSuccess || !ptr) { cudaGetLastError(); return OCTO_FMM_ECUDA; }
        if ((uintptr_t)ptr % ALIGN) return OCTO_FMM_ECUDA;
        sp.scratch = ptr;
    }
    if (!sp.h || !same_static_config(sp.key, c)) {
        // another configuration: a new handle over the same scratch (host memory only; the old one is drained first,
        // its kernels still read the array)
        if (sp.h) { octo_fmm* old = sp.h; sp.h = nullptr; if (octo_fmm_destroy(old) != OCTO_FMM_OK) return OCTO_FMM_ECUDA; }
        c.workspace = sp.scratch; c.workspace_bytes = STATIC_SCRATCH_BYTES;
        octo_fmm* h = nullptr;
        const int rc = create_internal(&c, 0, &h);
        if (rc != OCTO_FMM_OK) return rc;
        sp.h = h; sp.key = c;
    }
    octo_fmm* h = sp.h;
    int rc = octo_fmm_bind_outputs(h, L, Lcorr);
    if (rc != OCTO_FMM_OK) return rc;
    // the array keeps the last call's contents: the two flag words start at zero, every staged record of the grid is
    // rewritten by the staging kernel, and nothing outside the grid is read (TMA zero-fills / explicit in-grid tests)
    if (cudaMemsetAsync(h->flags, 0, 2 * sizeof(int), h->stream) != cudaSuccess) return OCTO_FMM_ECUDA;
    if ((rc = octo_fmm_set_moments(h, moments, com_off)) != OCTO_FMM_OK) return rc;
    return octo_fmm_interact(h);
}

int octo_fmm_static_status(int device)
{
    if (device < 0 || device >= MAX_DEVICES) return OCTO_FMM_EINVAL;
    std::lock_guard<std::mutex> guard(g_static_mu);
    if (!g_static[device].h) return OCTO_FMM_ESTATE;
    return octo_fmm_status(g_static[device].h);
}

}  // extern "C"

#include "solver.inl"
#include "tree.inl"
