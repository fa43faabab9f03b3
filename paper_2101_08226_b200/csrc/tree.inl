// tree.inl -- host logic and C ABI of the gravity solve on an adaptive oct-tree of 8^3 sub-grids (octo_fmm_tree_*,
// SURVEY 8(f) f3), included by octo_fmm.cu after solver.inl (it drives per-level octo_fmm handles
// through their internals, like the uniform solve).
//
// Levels: tree levels l = 0 .. depth-1 (dense [n_l]^3 lattices, n_l = n0 2^l, with kind[cell]); above level 0 the uniform
// multipole levels n0/2 .. 2 exactly as in the uniform solve.  Per tree level: a multipole handle (slab-fed kernel in
// MODE_TREE over the bricks that have work) if the level has refined cells, a monopole handle with the leaf-level list
// (tensor-core kernel over the tiles that hold leaves) if it has leaves.
// solve(): leaf moments + M2M bottom-up -> uniform levels up and down -> per tree level, coarsest first: stage, multipole
// step with the parent's expansion fused in, leaf-leaf sums, leaf finish (expansion at the centre + cross-level pairs).

namespace {

struct TreeLevel {
    int n[3];                   // extents of this level's arrays: a BOX of the level's lattice (multiples of 8)
    int lo[3];                  // lower corner of the box on the lattice (multiples of 8)
    int psh[3];                 // parent index in the parent level's arrays = (index >> 1) + psh
    double h;
    bool has_refined, has_leaf;
    unsigned char* kind;        // device [nz][ny][nx]
    unsigned char* nodeflag;    // device, per sub-grid
    double* lm;                 // device [cells] masked masses (leaf: m, else 0)
    double* raw;                // device [20][cells] (null on a level without refined cells)
    double* off;                // device [3][cells]
    octo_fmm* fmm;              // multipole handle (null without refined cells)
    octo_fmm* leaf;             // monopole handle, leaf-level list (null without leaves)
    int* m2l_tiles;  int n_m2l_tiles;     // bricks of the slab-fed kernel that have work
    int* p2p_tiles;  int n_p2p_tiles;     // 16 x 16 x 8 tiles of the tensor-core kernel that hold leaves
    std::vector<int> h_m2l_tiles, h_p2p_tiles;
    unsigned short* m2l_zmask;            // device, per listed brick: source layers that hold anything the brick can meet
    std::vector<unsigned short> h_m2l_zmask;
    int* ref_nodes;  int n_ref_nodes;     // device: the refined sub-grids of the level, x | y << 10 | z << 20 (box-local, sub-grid units)
    std::vector<int> h_ref_nodes;
    int* fin_nodes;  int n_fin_nodes;     // device: the sub-grids of the listed leaf tiles (whatever their kind): the cells the leaf
    std::vector<int> h_fin_nodes;         // finish visits; every other cell of the level's output is zero-filled by a memset
    unsigned char* brick_on;              // device [bricks of the dense enumeration]: 1 = the multipole step ran on this brick
    std::vector<unsigned char> h_brick_on;
    int btx, btz;                         // bricks per x-row and per z-column of that enumeration
    std::vector<unsigned char> h_nodeflag;
    // the multipole step and the leaf-leaf sums of a level depend on the upward pass only: they run on streams of their
    // own, side by side with those of the other levels; the L2L / leaf-finish chain on the caller's stream waits for them
    cudaStream_t s_m2l, s_leaf;
    cudaEvent_t ev_m2l, ev_leaf;
    bool m2l_on_main;                  // few bricks (a level near the top): its multipole step runs in the main stream's chain
    cudaEvent_t ev_lm;                 // on the leaf stream: this level's leaf masses (and the moments of its non-refined cells)
    cudaEvent_t ev_rdy;                // on the main stream: this level's raw moments and leaf masses are there (upward pass)
    cudaEvent_t ev_par;                // on the main stream: the PARENT level's expansions are complete (leaf finish may start)
    size_t cells() const { return (size_t)n[0] * n[1] * n[2]; }
};

struct TreePlan {
    std::vector<TreeLevel> lev;
    size_t bytes;
    bool ok;
};

inline bool tree_config_ok(const octo_fmm_tree_config* c)
{
    if (!c) return false;
    if (c->n0 < 8 || c->n0 > 2048 || (c->n0 & (c->n0 - 1))) return false;       // a power of two >= 8
    if (c->depth < 1 || c->depth > 12) return false;
    if (((long long)c->n0 << (c->depth - 1)) > (1 << 20)) return false;          // lattice indices stay far from 2^31
    if (!(c->h0 > 0.0) || !std::isfinite(c->h0)) return false;
    if (!(c->theta > 1.0 / 3.0 && c->theta < 1.0)) return false;
    return true;
}

octo_fmm_solver_config as_solver_config(const octo_fmm_tree_config& t)
{
    octo_fmm_solver_config s;
    std::memset(&s, 0, sizeof s);
    s.n = t.n0; s.h = t.h0; s.theta = t.theta; s.am_correction = t.am_correction; s.device = t.device; s.stream = t.stream;
    return s;
}

octo_fmm_config box_config(const octo_fmm_solver_config& sc, const int n[3], double h, int kind)
{
    octo_fmm_config c = level_config(sc, n[0], h, kind);
    for (int a = 0; a < 3; ++a) c.n[a] = n[a];
    return c;
}

// Topology checks, per-sub-grid flags, tile lists and the workspace size.  kind_host[l] = [nz][ny][nx] of level l's box on
// the HOST; box = null (every level is its whole lattice) or depth x 6 ints (lo_x, lo_y, lo_z, n_x, n_y, n_z).
TreePlan tree_plan(const octo_fmm_tree_config& cfg, const unsigned char* const* kind_host, const int* box)
{
    TreePlan P;
    P.ok = false;
    P.bytes = 0;
    const int D = cfg.depth;
    P.lev.resize(D);
    const octo_fmm_solver_config sc = as_solver_config(cfg);
    // kind of the sub-grid with LATTICE coordinates (I, J, K) of level l: absent outside the box
    auto node_kind = [&](int l, int I, int J, int K) -> unsigned char {
        const TreeLevel& L = P.lev[l];
        const int i = 8 * I - L.lo[0], j = 8 * J - L.lo[1], k = 8 * K - L.lo[2];
        if (i < 0 || j < 0 || k < 0 || i >= L.n[0] || j >= L.n[1] || k >= L.n[2]) return KIND_ABSENT;
        return kind_host[l][((size_t)k * L.n[1] + j) * L.n[0] + i];
    };
    for (int l = 0; l < D; ++l) {
        TreeLevel& L = P.lev[l];
        const long long lat = (long long)cfg.n0 << l;
        for (int a = 0; a < 3; ++a) {
            L.lo[a] = box ? box[6 * l + a] : 0;
            L.n[a] = box ? box[6 * l + 3 + a] : (int)lat;
            if (L.lo[a] < 0 || L.n[a] < 8 || (L.lo[a] % 8) || (L.n[a] % 8) || (long long)L.lo[a] + L.n[a] > lat || L.n[a] > 4096) return P;
            if (l == 0 && (L.lo[a] != 0 || L.n[a] != cfg.n0)) return P;      // level 0 is the whole lattice
            L.psh[a] = l > 0 ? L.lo[a] / 2 - P.lev[l - 1].lo[a] : 0;
        }
        L.h = cfg.h0 / (double)(1LL << l);
        L.fmm = nullptr; L.leaf = nullptr; L.kind = nullptr; L.nodeflag = nullptr; L.lm = nullptr; L.raw = nullptr; L.off = nullptr;
        L.m2l_tiles = nullptr; L.p2p_tiles = nullptr; L.n_m2l_tiles = 0; L.n_p2p_tiles = 0;
        L.brick_on = nullptr; L.btx = 0; L.btz = 0;
        L.m2l_zmask = nullptr;
        L.ref_nodes = nullptr; L.n_ref_nodes = 0; L.fin_nodes = nullptr; L.n_fin_nodes = 0;
        L.s_m2l = nullptr; L.s_leaf = nullptr; L.ev_m2l = nullptr; L.ev_leaf = nullptr; L.ev_par = nullptr; L.ev_rdy = nullptr; L.ev_lm = nullptr;
        const unsigned char* k = kind_host[l];
        if (!k) return P;
        L.has_refined = L.has_leaf = false;
        // kinds are constant over sub-grids, a cell exists iff its parent is refined, the last level has no refined cell
        for (int K = 0; K < L.n[2] / 8; ++K)
            for (int J = 0; J < L.n[1] / 8; ++J)
                for (int I = 0; I < L.n[0] / 8; ++I) {
                    const unsigned char v = k[((size_t)(8 * K) * L.n[1] + 8 * J) * L.n[0] + 8 * I];
                    if (v > 2) return P;
                    for (int c = 0; c < 8; ++c)
                        for (int b = 0; b < 8; ++b)
                            for (int a = 0; a < 8; ++a)
                                if (k[((size_t)(8 * K + c) * L.n[1] + 8 * J + b) * L.n[0] + 8 * I + a] != v) return P;
                    if (l == 0 && v == KIND_ABSENT) return P;
                    if (l == D - 1 && v == KIND_REFINED) return P;
                    if (l > 0) {
                        const unsigned char pv = node_kind(l - 1, (L.lo[0] / 8 + I) / 2, (L.lo[1] / 8 + J) / 2, (L.lo[2] / 8 + K) / 2);
                        if ((v != KIND_ABSENT) != (pv == KIND_REFINED)) return P;
                    }
                    L.has_refined |= v == KIND_REFINED;
                    L.has_leaf |= v == KIND_LEAF;
                }
        // every refined sub-grid of the level above has all its children inside this level's box
        if (l > 0) {
            const TreeLevel& U = P.lev[l - 1];
            for (int K = 0; K < U.n[2] / 8; ++K)
                for (int J = 0; J < U.n[1] / 8; ++J)
                    for (int I = 0; I < U.n[0] / 8; ++I) {
                        if (kind_host[l - 1][((size_t)(8 * K) * U.n[1] + 8 * J) * U.n[0] + 8 * I] != KIND_REFINED) continue;
                        for (int c = 0; c < 8; ++c)
                            if (node_kind(l, 2 * (U.lo[0] / 8 + I) + (c & 1), 2 * (U.lo[1] / 8 + J) + ((c >> 1) & 1),
                                          2 * (U.lo[2] / 8 + K) + (c >> 2)) == KIND_ABSENT)
                                return P;
                    }
        }
    }
    if (P.lev[D - 1].has_refined) return P;
    // flags: NODE_OWN_L = leaf sub-grid with a refined 26-neighbour; NODE_COARSE_NBR = the parent sub-grid has a leaf 26-neighbour
    for (int l = 0; l < D; ++l) {
        TreeLevel& L = P.lev[l];
        const int nnx = L.n[0] / 8, nny = L.n[1] / 8, nnz = L.n[2] / 8;
        const int gx0 = L.lo[0] / 8, gy0 = L.lo[1] / 8, gz0 = L.lo[2] / 8;
        L.h_nodeflag.assign((size_t)nnx * nny * nnz, 0);
        for (int K = 0; K < nnz; ++K)
            for (int J = 0; J < nny; ++J)
                for (int I = 0; I < nnx; ++I) {
                    if (node_kind(l, gx0 + I, gy0 + J, gz0 + K) == KIND_REFINED) L.h_ref_nodes.push_back(I | (J << 10) | (K << 20));
                    if (node_kind(l, gx0 + I, gy0 + J, gz0 + K) != KIND_LEAF) continue;
                    unsigned char f = 0;
                    for (int c = -1; c <= 1; ++c)
                        for (int b = -1; b <= 1; ++b)
                            for (int a = -1; a <= 1; ++a) {
                                if (node_kind(l, gx0 + I + a, gy0 + J + b, gz0 + K + c) == KIND_REFINED) f |= NODE_OWN_L;
                                if (l > 0 && node_kind(l - 1, (gx0 + I) / 2 + a, (gy0 + J) / 2 + b, (gz0 + K) / 2 + c) == KIND_LEAF)
                                    f |= NODE_COARSE_NBR;
                            }
                    L.h_nodeflag[((size_t)K * nny + J) * nnx + I] = f;
                }
        auto node_works = [&](int I, int J, int K) {   // local sub-grid: its cells take part in the multipole step of this level
            if (I >= nnx || J >= nny || K >= nnz) return false;
            const unsigned char v = node_kind(l, gx0 + I, gy0 + J, gz0 + K);
            return v == KIND_REFINED || (v == KIND_LEAF && (L.h_nodeflag[((size_t)K * nny + J) * nnx + I] & NODE_OWN_L));
        };
        // bricks of the slab-fed kernel: 16 x 8 x 3 cells, dense enumeration t = (ty * tiles_x + tx) * tiles_z + tz
        if (L.has_refined) {
            const int tx_n = (L.n[0] + TILE_X - 1) / TILE_X, ty_n = (L.n[1] + TILE_Y - 1) / TILE_Y, tz_n = (L.n[2] + TILE_Z - 1) / TILE_Z;
            std::vector<std::pair<double, int>> weighted;
            for (int ty = 0; ty < ty_n; ++ty)
                for (int tx = 0; tx < tx_n; ++tx)
                    for (int tz = 0; tz < tz_n; ++tz) {
                        // estimated work of the brick: its cells in refined sub-grids count fully, those in leaf sub-grids next
                        // to refined ones about a fifth (most of their list entries are skipped)
                        double weight = 0.0;
                        const int z0 = tz * TILE_Z, z1 = std::min(z0 + TILE_Z, L.n[2]) - 1;
                        for (int K = z0 / 8; K <= z1 / 8; ++K)
                            for (int I = (tx * TILE_X) / 8; I <= std::min(tx * TILE_X + TILE_X - 1, L.n[0] - 1) / 8; ++I) {
                                if (!node_works(I, (ty * TILE_Y) / 8, K)) continue;
                                const int layers = std::min(z1, 8 * K + 7) - std::max(z0, 8 * K) + 1;
                                const bool refined = node_kind(l, gx0 + I, gy0 + (ty * TILE_Y) / 8, gz0 + K) == KIND_REFINED;
                                weight += (refined ? 1.0 : 0.2) * 64.0 * layers;
                            }
                        if (weight <= 0.0) continue;
                        // a brick of leaf cells only has work if a refined cell lies within the lists' reach of it (the
                        // sub-grid flag says "within a sub-grid": 8 cells, and a sub-grid has 2 x 1 x 3 bricks)
                        bool near_refined = false;
                        const int xa = tx * TILE_X - REACH_MAX, xb = std::min(tx * TILE_X + TILE_X, L.n[0]) - 1 + REACH_MAX;
                        const int ya = ty * TILE_Y - REACH_MAX, yb = std::min(ty * TILE_Y + TILE_Y, L.n[1]) - 1 + REACH_MAX;
                        const int za = z0 - REACH_MAX, zb = z1 + REACH_MAX;
                        for (int K = floor_div8(za); K <= floor_div8(zb) && !near_refined; ++K)
                            for (int J = floor_div8(ya); J <= floor_div8(yb) && !near_refined; ++J)
                                for (int I = floor_div8(xa); I <= floor_div8(xb) && !near_refined; ++I)
                                    near_refined = I >= 0 && J >= 0 && K >= 0 && I < nnx && J < nny && K < nnz &&
                                                   node_kind(l, gx0 + I, gy0 + J, gz0 + K) == KIND_REFINED;
                        if (!near_refined) continue;
                        weighted.push_back(std::make_pair(-weight, (ty * tx_n + tx) * tz_n + tz));
                    }
            L.btx = tx_n; L.btz = tz_n;
            L.h_brick_on.assign((size_t)tx_n * ty_n * tz_n, 0);
            for (const auto& wt : weighted) L.h_brick_on[wt.second] = 1;
            // heaviest bricks first: the persistent CTAs take the list round-robin, so that every CTA gets its share of the
            // bricks that are full of refined cells instead of whoever comes first in lattice order getting three of them
            std::sort(weighted.begin(), weighted.end());
            for (const auto& wt : weighted) L.h_m2l_tiles.push_back(wt.second);
            // per brick, the source layers worth loading: a brick with refined targets meets every cell that exists, a
            // brick of leaves only refined ones; layers whose 26 x 18 footprint holds none are left out (bit i = layer
            // k0 - REACH_MAX + i).  Kinds are constant over sub-grids, so sub-grids are what is tested.
            for (const int tile : L.h_m2l_tiles) {
                const int tz = tile % tz_n, tx = (tile / tz_n) % tx_n, ty = tile / (tz_n * tx_n);
                const int x0 = tx * TILE_X, y0 = ty * TILE_Y, k0 = tz * TILE_Z;
                bool refined_targets = false;
                for (int K = k0 / 8; K <= std::min(k0 + TILE_Z - 1, L.n[2] - 1) / 8 && !refined_targets; ++K)
                    for (int I = x0 / 8; I <= std::min(x0 + TILE_X - 1, L.n[0] - 1) / 8 && !refined_targets; ++I)
                        refined_targets = node_kind(l, gx0 + I, gy0 + y0 / 8, gz0 + K) == KIND_REFINED;
                unsigned short mask = 0;
                for (int i = 0; i < TILE_Z + 2 * REACH_MAX; ++i) {
                    const int zz = k0 - REACH_MAX + i;
                    if (zz < 0 || zz >= L.n[2]) continue;
                    bool any = false;
                    for (int J = floor_div8(y0 - REACH_MAX); J <= floor_div8(y0 + TILE_Y - 1 + REACH_MAX) && !any; ++J)
                        for (int I = floor_div8(x0 - REACH_MAX); I <= floor_div8(x0 + TILE_X - 1 + REACH_MAX) && !any; ++I) {
                            if (I < 0 || J < 0 || I >= nnx || J >= nny) continue;
                            const unsigned char v = node_kind(l, gx0 + I, gy0 + J, gz0 + zz / 8);
                            any = refined_targets ? v != KIND_ABSENT : v == KIND_REFINED;
                        }
                    if (any) mask |= (unsigned short)(1u << i);
                }
                L.h_m2l_zmask.push_back(mask);
            }
        }
        // tiles of the tensor-core leaf kernel: 16 x 16 x 8 cells, b = (tz * by + ty) * bx + tx
        if (L.has_leaf) {
            const int bx = (L.n[0] + MT_X - 1) / MT_X, by = (L.n[1] + MT_Y - 1) / MT_Y, bz = (L.n[2] + DT_Z - 1) / DT_Z;
            for (int tz = 0; tz < bz; ++tz)
                for (int ty = 0; ty < by; ++ty)
                    for (int tx = 0; tx < bx; ++tx) {
                        bool work = false;
                        for (int J = 2 * ty; J <= std::min(2 * ty + 1, nny - 1) && !work; ++J)
                            for (int I = 2 * tx; I <= std::min(2 * tx + 1, nnx - 1) && !work; ++I)
                                work = node_kind(l, gx0 + I, gy0 + J, gz0 + tz) == KIND_LEAF;
                        if (!work) continue;
                        L.h_p2p_tiles.push_back((tz * by + ty) * bx + tx);
                        for (int J = 2 * ty; J <= std::min(2 * ty + 1, nny - 1); ++J)
                            for (int I = 2 * tx; I <= std::min(2 * tx + 1, nnx - 1); ++I) L.h_fin_nodes.push_back(I | (J << 10) | (tz << 20));
                    }
        }
        L.n_m2l_tiles = (int)L.h_m2l_tiles.size();
        L.n_p2p_tiles = (int)L.h_p2p_tiles.size();
        // workspace of this level
        const size_t nc = L.cells();
        P.bytes += align_up(nc) + align_up((size_t)nnx * nny * nnz) + align_up(nc * 8);           // kind, nodeflag, lm
        L.n_ref_nodes = (int)L.h_ref_nodes.size();
        L.n_fin_nodes = (int)L.h_fin_nodes.size();
        P.bytes += align_up((size_t)L.n_m2l_tiles * 4 + 4) + align_up((size_t)L.n_m2l_tiles * 2 + 4) + align_up((size_t)L.n_p2p_tiles * 4 + 4) + align_up(L.h_brick_on.size() + 4) +
                   align_up((size_t)L.n_ref_nodes * 4 + 4) + align_up((size_t)L.n_fin_nodes * 4 + 4);
        if (L.has_refined) {
            octo_fmm_config mc = box_config(sc, L.n, L.h, OCTO_FMM_MULTIPOLE);
            P.bytes += sizes_of(mc, CF_ANY_SIZE).total + align_up(nc * 20 * 8) + align_up(nc * 3 * 8);
        }
        if (L.has_leaf) {
            octo_fmm_config lc = box_config(sc, L.n, L.h, OCTO_FMM_MONOPOLE);
            P.bytes += sizes_of(lc, CF_LEAF_LIST).total;
        }
    }
    // the uniform levels above level 0
    double h = cfg.h0;
    for (int n = cfg.n0 / 2; n >= 2; n /= 2) {
        h *= 2.0;
        octo_fmm_config mc = level_config(sc, n, h, OCTO_FMM_MULTIPOLE);
        const size_t nc = (size_t)n * n * n;
        P.bytes += sizes_of(mc, CF_ANY_SIZE).total + align_up(nc * 20 * 8) + align_up(nc * 3 * 8);
    }
    P.bytes += ALIGN;      // pair counters
    P.ok = true;
    return P;
}

}  // namespace

struct octo_fmm_tree {
    octo_fmm_tree_config cfg;
    std::vector<TreeLevel> lev;        // tree levels, coarsest first
    std::vector<SolverLevel> up;       // uniform levels n0/2, ..., 2
    unsigned long long* counts;        // device [3]: m2l, p2p, cross
    cudaStream_t stream;               // the solve's own main stream (high priority): upward pass, uniform levels, L2L chain
    cudaStream_t pool_m2l[3], pool_leaf[2];   // the levels share a few side streams (see octo_fmm_tree_create)
    cudaStream_t s_d2h;                // octo_fmm_tree_solve_host: the copies out (created on first use)
    cudaStream_t user;                 // the caller's stream (cfg.stream): a solve starts after and is joined into it
    cudaEvent_t ev_user;               // hand-over between the two
    cudaEvent_t ev_up;                 // a solve has begun on the main stream (the side streams start behind it)
    cudaEvent_t ev_top_rdy, ev_top_m2l;   // the finest uniform level: its moments are there / its multipole step is done
    bool solved;
};

extern "C" {

size_t octo_fmm_tree_workspace_bytes(const octo_fmm_tree_config* cfg, const unsigned char* const* kind_host, const int* box)
{
    if (!tree_config_ok(cfg) || !kind_host) return 0;
    const TreePlan P = tree_plan(*cfg, kind_host, box);
    return P.ok ? P.bytes : 0;
}

int octo_fmm_tree_destroy(octo_fmm_tree_t* t)
{
    if (!t) return OCTO_FMM_EINVAL;
    int rc = OCTO_FMM_OK;
    for (TreeLevel& l : t->lev) {
        if (l.fmm && octo_fmm_destroy(l.fmm) != OCTO_FMM_OK) rc = OCTO_FMM_ECUDA;
        if (l.leaf && octo_fmm_destroy(l.leaf) != OCTO_FMM_OK) rc = OCTO_FMM_ECUDA;
    }
    for (SolverLevel& l : t->up)
        if (l.fmm && octo_fmm_destroy(l.fmm) != OCTO_FMM_OK) rc = OCTO_FMM_ECUDA;
    for (TreeLevel& l : t->lev) {
        if (l.ev_m2l) cudaEventDestroy(l.ev_m2l);
        if (l.ev_leaf) cudaEventDestroy(l.ev_leaf);
        if (l.ev_par) cudaEventDestroy(l.ev_par);
        if (l.ev_rdy) cudaEventDestroy(l.ev_rdy);
        if (l.ev_lm) cudaEventDestroy(l.ev_lm);
    }
    if (t->ev_up) cudaEventDestroy(t->ev_up);
    if (t->ev_top_rdy) cudaEventDestroy(t->ev_top_rdy);
    if (t->ev_top_m2l) cudaEventDestroy(t->ev_top_m2l);
    if (t->ev_user) cudaEventDestroy(t->ev_user);
    for (cudaStream_t& q : t->pool_m2l) if (q) cudaStreamDestroy(q);
    for (cudaStream_t& q : t->pool_leaf) if (q) cudaStreamDestroy(q);
    if (t->s_d2h) cudaStreamDestroy(t->s_d2h);
    if (t->stream) cudaStreamDestroy(t->stream);
    delete t;
    return rc;
}

int octo_fmm_tree_create(const octo_fmm_tree_config* cfg, const unsigned char* const* kind_host, const int* box, octo_fmm_tree_t** out)
{
    if (!out) return OCTO_FMM_EINVAL;
    *out = nullptr;
    if (!tree_config_ok(cfg) || !kind_host) return OCTO_FMM_EINVAL;
    TreePlan P = tree_plan(*cfg, kind_host, box);
    if (!P.ok) return OCTO_FMM_EINVAL;
    if (!cfg->workspace || cfg->workspace_bytes < P.bytes || ((uintptr_t)cfg->workspace % ALIGN)) return OCTO_FMM_EINVAL;
    if (cudaSetDevice(cfg->device) != cudaSuccess) return OCTO_FMM_ECUDA;
    octo_fmm_tree* t = new (std::nothrow) octo_fmm_tree();
    if (!t) return OCTO_FMM_ENOMEM;
    t->cfg = *cfg;
    t->user = (cudaStream_t)cfg->stream;
    t->stream = nullptr;
    t->solved = false;
    t->ev_up = nullptr; t->ev_user = nullptr; t->ev_top_rdy = nullptr; t->ev_top_m2l = nullptr;
    t->lev = std::move(P.lev);
    // Streams.  The multipole steps of the levels are long CTAs that fill every SM (one per SM, 100 us each); whatever
    // else a solve launches is short and must not queue behind them: it runs on streams of the HIGHEST priority (the
    // block scheduler hands a freed SM to them first), the multipole steps on streams of the lowest.
    int prio_least = 0, prio_greatest = 0;
    if (cudaDeviceGetStreamPriorityRange(&prio_least, &prio_greatest) != cudaSuccess ||
        cudaStreamCreateWithPriority(&t->stream, cudaStreamNonBlocking, prio_greatest) != cudaSuccess ||
        cudaEventCreateWithFlags(&t->ev_user, cudaEventDisableTiming) != cudaSuccess) { octo_fmm_tree_destroy(t); return OCTO_FMM_ECUDA; }
    // FEW side streams, shared by the levels (three for the multipole steps, leaf stream l % 2): a device runs only a
    // handful of hardware work queues (8 by default), and streams beyond that number alias onto the same queue -- with one
    // stream pair per level (19 streams at 9 levels) a level's multipole step started only when ANOTHER level's had
    // ended.
    for (cudaStream_t& q : t->pool_m2l)
        if (cudaStreamCreateWithPriority(&q, cudaStreamNonBlocking, prio_least) != cudaSuccess) { octo_fmm_tree_destroy(t); return OCTO_FMM_ECUDA; }
    // (the leaf streams one step below the main stream: the short L2L chain must not queue behind a leaf finish)
    const int prio_leaf = prio_greatest < prio_least ? prio_greatest + 1 : prio_greatest;
    for (cudaStream_t& q : t->pool_leaf)
        if (cudaStreamCreateWithPriority(&q, cudaStreamNonBlocking, prio_leaf) != cudaSuccess) { octo_fmm_tree_destroy(t); return OCTO_FMM_ECUDA; }
    // multipole streams: the levels with at least one brick per SM take turns on the three, SHALLOWEST first (the L2L chain
    // goes down the tree: what is left when the last multipole step ends is then one level's L2L and two leaf finishes);
    // the small levels at the top run inside the main stream's chain, which needs them first anyway
    int big_rank = 0;
    std::vector<int> m2l_stream(t->lev.size(), -1);
    for (size_t l = 0; l < t->lev.size(); ++l)
        if (t->lev[l].n_m2l_tiles >= 148) m2l_stream[l] = big_rank++ % 3;
    octo_fmm_solver_config sc = as_solver_config(*cfg);
    sc.stream = t->stream;
    char* w = (char*)cfg->workspace;
    cudaStream_t st = t->stream;
    int rc = OCTO_FMM_OK;
    for (size_t l = 0; l < t->lev.size() && rc == OCTO_FMM_OK; ++l) {
        TreeLevel& L = t->lev[l];
        const size_t nc = L.cells(), nn = (size_t)(L.n[0] / 8) * (L.n[1] / 8) * (L.n[2] / 8);
        L.kind = (unsigned char*)w; w += align_up(nc);
        L.nodeflag = (unsigned char*)w; w += align_up(nn);
        L.lm = (double*)w; w += align_up(nc * 8);
        L.m2l_tiles = (int*)w; w += align_up((size_t)L.n_m2l_tiles * 4 + 4);
        L.p2p_tiles = (int*)w; w += align_up((size_t)L.n_p2p_tiles * 4 + 4);
        L.m2l_zmask = (unsigned short*)w; w += align_up((size_t)L.n_m2l_tiles * 2 + 4);
        L.brick_on = (unsigned char*)w; w += align_up(L.h_brick_on.size() + 4);
        L.ref_nodes = (int*)w; w += align_up((size_t)L.n_ref_nodes * 4 + 4);
        L.fin_nodes = (int*)w; w += align_up((size_t)L.n_fin_nodes * 4 + 4);
        if (cudaMemcpyAsync(L.kind, kind_host[l], nc, cudaMemcpyHostToDevice, st) != cudaSuccess ||
            cudaMemcpyAsync(L.nodeflag, L.h_nodeflag.data(), nn, cudaMemcpyHostToDevice, st) != cudaSuccess ||
            (L.n_m2l_tiles && cudaMemcpyAsync(L.m2l_tiles, L.h_m2l_tiles.data(), (size_t)L.n_m2l_tiles * 4, cudaMemcpyHostToDevice, st) != cudaSuccess) ||
            (L.n_m2l_tiles && cudaMemcpyAsync(L.m2l_zmask, L.h_m2l_zmask.data(), (size_t)L.n_m2l_tiles * 2, cudaMemcpyHostToDevice, st) != cudaSuccess) ||
            (L.n_p2p_tiles && cudaMemcpyAsync(L.p2p_tiles, L.h_p2p_tiles.data(), (size_t)L.n_p2p_tiles * 4, cudaMemcpyHostToDevice, st) != cudaSuccess) ||
            (!L.h_brick_on.empty() && cudaMemcpyAsync(L.brick_on, L.h_brick_on.data(), L.h_brick_on.size(), cudaMemcpyHostToDevice, st) != cudaSuccess) ||
            (L.n_ref_nodes && cudaMemcpyAsync(L.ref_nodes, L.h_ref_nodes.data(), (size_t)L.n_ref_nodes * 4, cudaMemcpyHostToDevice, st) != cudaSuccess) ||
            (L.n_fin_nodes && cudaMemcpyAsync(L.fin_nodes, L.h_fin_nodes.data(), (size_t)L.n_fin_nodes * 4, cudaMemcpyHostToDevice, st) != cudaSuccess)) {
            rc = OCTO_FMM_ECUDA;
            break;
        }
        L.m2l_on_main = m2l_stream[l] < 0;
        L.s_m2l = L.m2l_on_main ? t->stream : t->pool_m2l[m2l_stream[l]];
        L.s_leaf = t->pool_leaf[l % 2];
        if (cudaEventCreateWithFlags(&L.ev_rdy, cudaEventDisableTiming) != cudaSuccess ||
            cudaEventCreateWithFlags(&L.ev_lm, cudaEventDisableTiming) != cudaSuccess ||
            cudaEventCreateWithFlags(&L.ev_m2l, cudaEventDisableTiming) != cudaSuccess ||
            cudaEventCreateWithFlags(&L.ev_leaf, cudaEventDisableTiming) != cudaSuccess ||
            cudaEventCreateWithFlags(&L.ev_par, cudaEventDisableTiming) != cudaSuccess) { rc = OCTO_FMM_ECUDA; break; }
        if (L.has_refined) {
            octo_fmm_config mc = box_config(sc, L.n, L.h, OCTO_FMM_MULTIPOLE);
            mc.stream = L.s_m2l;
            mc.workspace = w; mc.workspace_bytes = sizes_of(mc, CF_ANY_SIZE).total; w += mc.workspace_bytes;
            L.raw = (double*)w; w += align_up(nc * 20 * 8);
            L.off = (double*)w; w += align_up(nc * 3 * 8);
            rc = create_internal(&mc, CF_ANY_SIZE, &L.fmm);
            if (rc != OCTO_FMM_OK) break;
            L.fmm->kernel = 0;                 // the slab-fed kernel (MODE_TREE), whatever the size of the level
            L.fmm->tree_kind = L.kind;
            L.fmm->tile_list = L.m2l_tiles;
            L.fmm->tile_zmask = L.m2l_zmask;
            L.fmm->tile_count = L.n_m2l_tiles;
            // what never changes from solve to solve is written here, once: the zeros of the moments and offsets of the
            // cells that are not refined (a leaf is a point mass at its centre) and their staged records, with every cell's
            // kind in the padding slot (tree.cuh: tree_leaf_moments_kernel)
            if (cudaMemsetAsync(L.raw, 0, nc * 20 * 8, st) != cudaSuccess || cudaMemsetAsync(L.off, 0, nc * 3 * 8, st) != cudaSuccess) {
                rc = OCTO_FMM_ECUDA;
                break;
            }
            tree_stage_init_kernel<<<(unsigned)((nc + 255) / 256), 256, 0, st>>>(L.kind, L.fmm->src, L.n[0], L.n[1], L.n[2],
                                                                              L.fmm->cfg.am_correction);
            if (cudaGetLastError() != cudaSuccess) { rc = OCTO_FMM_ECUDA; break; }
        }
        if (L.has_leaf) {
            octo_fmm_config lc = box_config(sc, L.n, L.h, OCTO_FMM_MONOPOLE);
            lc.stream = L.s_leaf;
            lc.workspace = w; lc.workspace_bytes = sizes_of(lc, CF_LEAF_LIST).total; w += lc.workspace_bytes;
            rc = create_internal(&lc, CF_LEAF_LIST, &L.leaf);
            if (rc != OCTO_FMM_OK) break;
            L.leaf->tile_list = L.p2p_tiles;
            L.leaf->tile_count = L.n_p2p_tiles;
        }
    }
    double h = cfg->h0;
    for (int n = cfg->n0 / 2; n >= 2 && rc == OCTO_FMM_OK; n /= 2) {
        h *= 2.0;
        SolverLevel l;
        l.n = n; l.h = h; l.fmm = nullptr; l.fmm2 = nullptr; l.raw2 = nullptr;
        octo_fmm_config mc = level_config(sc, n, h, OCTO_FMM_MULTIPOLE);
        const size_t nc = (size_t)n * n * n;
        l.ws_bytes = sizes_of(mc, CF_ANY_SIZE).total;
        mc.workspace = w; mc.workspace_bytes = l.ws_bytes; w += l.ws_bytes;
        l.raw = (double*)w; w += align_up(nc * 20 * 8);
        l.off = (double*)w; w += align_up(nc * 3 * 8);
        rc = create_internal(&mc, CF_ANY_SIZE, &l.fmm);
        t->up.push_back(l);
    }
    t->counts = (unsigned long long*)w;
    if (rc == OCTO_FMM_OK && (cudaEventCreateWithFlags(&t->ev_up, cudaEventDisableTiming) != cudaSuccess ||
                              cudaEventCreateWithFlags(&t->ev_top_rdy, cudaEventDisableTiming) != cudaSuccess ||
                              cudaEventCreateWithFlags(&t->ev_top_m2l, cudaEventDisableTiming) != cudaSuccess)) rc = OCTO_FMM_ECUDA;
    // the topology arrays were copied from pageable host memory: make sure they have left it before returning
    if (rc == OCTO_FMM_OK && cudaStreamSynchronize(st) != cudaSuccess) rc = OCTO_FMM_ECUDA;
    if (rc != OCTO_FMM_OK) { octo_fmm_tree_destroy(t); return rc; }
    for (TreeLevel& L : t->lev) { L.h_m2l_tiles.clear(); L.h_p2p_tiles.clear(); L.h_nodeflag.clear(); L.h_brick_on.clear(); L.h_ref_nodes.clear(); L.h_fin_nodes.clear(); L.h_m2l_zmask.clear(); }
    *out = t;
    return OCTO_FMM_OK;
}

// rhs2 (second right-hand side, L81-83): the sources are d(mass)/dt, expanded about the centres the last solve left in the
// off arrays (M2M with GIVEN centres), no correction; out[l] is then [cells]: the potential only.
// hand-over between the caller's stream and the solve's main stream
static int tree_enter(octo_fmm_tree_t* t)
{
    return cudaEventRecord(t->ev_user, t->user) == cudaSuccess && cudaStreamWaitEvent(t->stream, t->ev_user, 0) == cudaSuccess
               ? OCTO_FMM_OK : OCTO_FMM_ECUDA;
}
static int tree_leave(octo_fmm_tree_t* t)
{
    return cudaEventRecord(t->ev_user, t->stream) == cudaSuccess && cudaStreamWaitEvent(t->user, t->ev_user, 0) == cudaSuccess
               ? OCTO_FMM_OK : OCTO_FMM_ECUDA;
}

static int tree_solve_impl(octo_fmm_tree_t* t, const double* const* mass, double* const* out, bool count, bool rhs2 = false)
{
    const int D = (int)t->lev.size();
    cudaStream_t st = t->stream;
    int rc;
    if ((rc = tree_enter(t)) != OCTO_FMM_OK) return rc;
    // the level handles run without the correction for the second right-hand side (it belongs to the force, L127)
    struct CorrGuard {
        octo_fmm_tree_t* t; bool on; std::vector<int> keep;
        CorrGuard(octo_fmm_tree_t* t_, bool on_) : t(t_), on(on_) {
            if (!on) return;
            for (TreeLevel& l : t->lev) { keep.push_back(l.fmm ? l.fmm->cfg.am_correction : 0); if (l.fmm) l.fmm->cfg.am_correction = 0; }
            for (SolverLevel& l : t->up) { keep.push_back(l.fmm->cfg.am_correction); l.fmm->cfg.am_correction = 0; }
        }
        ~CorrGuard() {
            if (!on) return;
            size_t i = 0;
            for (TreeLevel& l : t->lev) { if (l.fmm) l.fmm->cfg.am_correction = keep[i]; ++i; }
            for (SolverLevel& l : t->up) l.fmm->cfg.am_correction = keep[i++];
        }
    } corr_guard(t, rhs2);
    // ---- upward pass.  The leaf masses of a level depend on nothing: every level writes them on its leaf stream, side by
    //      side (and its leaf-leaf sums follow there); the main stream carries only the M2M chain, finest level first ----
    if (cudaEventRecord(t->ev_up, st) != cudaSuccess) return OCTO_FMM_ECUDA;       // the solve has begun
    for (int l = D - 1; l >= 0; --l) {
        TreeLevel& L = t->lev[l];
        const long long nc = (long long)L.cells();
        if (cudaStreamWaitEvent(L.s_leaf, t->ev_up, 0) != cudaSuccess) return OCTO_FMM_ECUDA;
        // (the cells that are not refined: mass into raw, lm and the staged record; their zeros date from create())
        tree_leaf_moments_kernel<<<(unsigned)((nc + 255) / 256), 256, 0, L.s_leaf>>>(L.kind, mass[l], L.raw, L.lm, L.fmm ? L.fmm->src : nullptr,
                                                                                     L.n[0], L.n[1], nc);
        if (cudaGetLastError() != cudaSuccess) return OCTO_FMM_ECUDA;
        if (cudaEventRecord(L.ev_lm, L.s_leaf) != cudaSuccess) return OCTO_FMM_ECUDA;
        // the level's output: zero wherever the leaf finish does not go (it visits the sub-grids of the leaf tiles only)
        if (cudaMemsetAsync(out[l], 0, (size_t)nc * (rhs2 ? 1 : 4) * sizeof(double), L.s_leaf) != cudaSuccess) return OCTO_FMM_ECUDA;
    }
    for (int l = D - 1; l >= 0; --l) {
        TreeLevel& L = t->lev[l];
        if (L.has_refined) {
            TreeLevel& F = t->lev[l + 1];
            if (cudaStreamWaitEvent(st, F.ev_lm, 0) != cudaSuccess) return OCTO_FMM_ECUDA;      // the children that are leaves
            ChildBox cb;
            for (int a = 0; a < 3; ++a) { cb.n[a] = F.n[a]; cb.sh[a] = -2 * F.psh[a]; }
            cb.pkind = L.kind;
            cb.nodes = L.ref_nodes;
            const dim3 blocks(4u * (unsigned)L.n_ref_nodes);          // the refined sub-grids only: 512 parents = 4 blocks each
            if (rhs2) {
                if (F.raw) m2m_kernel<false, true, true><<<blocks, 128, 0, st>>>(F.raw, F.off, L.raw, L.off, L.n[0], L.n[1], L.n[2], F.h, cb);
                else       m2m_kernel<true, true, true><<<blocks, 128, 0, st>>>(F.lm, nullptr, L.raw, L.off, L.n[0], L.n[1], L.n[2], F.h, cb);
            } else {
                if (F.raw) m2m_kernel<false, false, true><<<blocks, 128, 0, st>>>(F.raw, F.off, L.raw, L.off, L.n[0], L.n[1], L.n[2], F.h, cb);
                else       m2m_kernel<true, false, true><<<blocks, 128, 0, st>>>(F.lm, nullptr, L.raw, L.off, L.n[0], L.n[1], L.n[2], F.h, cb);
            }
            if (cudaGetLastError() != cudaSuccess) return OCTO_FMM_ECUDA;
        }
        // this level's moments are complete (refined cells: M2M; the others: its leaf masses): its multipole step needs
        // nothing of the coarser levels and may start now
        if (cudaStreamWaitEvent(st, L.ev_lm, 0) != cudaSuccess) return OCTO_FMM_ECUDA;
        if (cudaEventRecord(L.ev_rdy, st) != cudaSuccess) return OCTO_FMM_ECUDA;
    }
    // ---- side by side: staging + multipole step per level (its own level only; the parent's expansion comes in the chain
    //      below), and the leaf-leaf point-mass sums ----
    auto multipole_step = [&](TreeLevel& L) -> int {
        if (cudaStreamWaitEvent(L.s_m2l, L.ev_rdy, 0) != cudaSuccess) return OCTO_FMM_ECUDA;
        // staging: the cells that are not refined were staged with their masses (tree_leaf_moments_kernel); the refined ones
        // got their moments from M2M just now
        int r;
        if (cudaMemsetAsync(L.fmm->flags + 1, 0, sizeof(int), L.s_m2l) != cudaSuccess) return OCTO_FMM_ECUDA;
        if (L.n_ref_nodes > 0) {
            tree_stage_refined_kernel<<<4u * (unsigned)L.n_ref_nodes, 128, 0, L.s_m2l>>>(L.raw, L.off, L.fmm->src, L.n[0], L.n[1], L.n[2], L.fmm->cfg.h,
                                                                                     L.fmm->flags, L.fmm->cfg.am_correction, L.ref_nodes);
            if (cudaGetLastError() != cudaSuccess) return OCTO_FMM_ECUDA;
        }
        L.fmm->state = 1;
        clear_parent(L.fmm);
        if ((r = octo_fmm_interact(L.fmm)) != OCTO_FMM_OK) return r;
        return cudaEventRecord(L.ev_m2l, L.s_m2l) == cudaSuccess ? OCTO_FMM_OK : OCTO_FMM_ECUDA;
    };
    for (int l = 0; l < D; ++l) {
        TreeLevel& L = t->lev[l];
        if (L.fmm && L.n_m2l_tiles > 0 && !L.m2l_on_main && (rc = multipole_step(L)) != OCTO_FMM_OK) return rc;
        if (L.leaf) {
            // (behind this level's leaf masses in the same stream)
            if ((rc = octo_fmm_set_moments(L.leaf, L.lm, nullptr)) != OCTO_FMM_OK) return rc;
            double* const keep = L.leaf->outL;
            if (!rhs2) L.leaf->outL = out[l];          // second right-hand side: the four sums go to the handle's own buffer
            rc = octo_fmm_interact(L.leaf);
            L.leaf->outL = keep;
            if (rc != OCTO_FMM_OK) return rc;
            if (cudaEventRecord(L.ev_leaf, L.s_leaf) != cudaSuccess) return OCTO_FMM_ECUDA;
        }
    }
    // ---- meanwhile on the caller's stream: the uniform levels above level 0 (the whole lattice), up ... ----
    const bool top_early = t->up.size() > 1 && t->up[0].fmm->kernel == 0;
    for (size_t lv = 0; lv < t->up.size(); ++lv) {
        SolverLevel& l = t->up[lv];
        const dim3 blocks((unsigned)((l.n + 127) / 128), (unsigned)l.n, (unsigned)l.n);
        if (lv == 0) {
            TreeLevel& B = t->lev[0];
            if (rhs2) {
                if (B.raw) m2m_kernel<false, true><<<blocks, 128, 0, st>>>(B.raw, B.off, l.raw, l.off, l.n, l.n, l.n, B.h);
                else       m2m_kernel<true, true><<<blocks, 128, 0, st>>>(B.lm, nullptr, l.raw, l.off, l.n, l.n, l.n, B.h);
            } else {
                if (B.raw) m2m_kernel<false><<<blocks, 128, 0, st>>>(B.raw, B.off, l.raw, l.off, l.n, l.n, l.n, B.h);
                else       m2m_kernel<true><<<blocks, 128, 0, st>>>(B.lm, nullptr, l.raw, l.off, l.n, l.n, l.n, B.h);
            }
        } else if (rhs2) {
            m2m_kernel<false, true><<<blocks, 128, 0, st>>>(t->up[lv - 1].raw, t->up[lv - 1].off, l.raw, l.off, l.n, l.n, l.n, t->up[lv - 1].h);
        } else {
            m2m_kernel<false><<<blocks, 128, 0, st>>>(t->up[lv - 1].raw, t->up[lv - 1].off, l.raw, l.off, l.n, l.n, l.n, t->up[lv - 1].h);
        }
        if (cudaGetLastError() != cudaSuccess) return OCTO_FMM_ECUDA;
        // The finest uniform level, when it is big enough for the slab-fed kernel (32^3 above a 64^3 base: 88 bricks, 110 us),
        // does not wait for its turn in the chain: its multipole step needs nothing but its own moments and starts now, on a
        // leaf stream (high priority: the chain will want it before the bricks of the tree levels that already fill the SMs),
        // while the main stream goes up to the root and comes down again; the L2L it had as an epilogue becomes a pass of its
        // own in the chain (12 us)
        if (lv == 0 && top_early) {
            cudaStream_t sx = t->pool_leaf[1];
            if (cudaEventRecord(t->ev_top_rdy, st) != cudaSuccess || cudaStreamWaitEvent(sx, t->ev_top_rdy, 0) != cudaSuccess) return OCTO_FMM_ECUDA;
            struct Lend { octo_fmm* h; cudaStream_t keep; Lend(octo_fmm* h_, cudaStream_t s) : h(h_), keep(h_->stream) { h->stream = s; } ~Lend() { h->stream = keep; } } lend(l.fmm, sx);
            if ((rc = octo_fmm_set_moments(l.fmm, l.raw, l.off)) != OCTO_FMM_OK) return rc;
            clear_parent(l.fmm);
            if ((rc = octo_fmm_interact(l.fmm)) != OCTO_FMM_OK) return rc;
            if (cudaEventRecord(t->ev_top_m2l, sx) != cudaSuccess) return OCTO_FMM_ECUDA;
        }
    }
    // ---- ... and down, as in the uniform solve ----
    for (int lv = (int)t->up.size() - 1; lv >= 0; --lv) {
        SolverLevel& l = t->up[lv];
        const bool has_parent = lv < (int)t->up.size() - 1;
        const bool early = lv == 0 && top_early;
        const bool fused = has_parent && l.fmm->kernel == 0 && !early;
        if (early) {
            if (cudaStreamWaitEvent(st, t->ev_top_m2l, 0) != cudaSuccess) return OCTO_FMM_ECUDA;
        } else {
            if ((rc = octo_fmm_set_moments(l.fmm, l.raw, l.off)) != OCTO_FMM_OK) return rc;
            if (fused) set_parent(l.fmm, t->up[lv + 1]);
            rc = octo_fmm_interact(l.fmm);
            if (fused) clear_parent(l.fmm);
            if (rc != OCTO_FMM_OK) return rc;
        }
        const dim3 blocks((unsigned)((l.n + 127) / 128), (unsigned)l.n, (unsigned)l.n);
        if (!has_parent)
            l2l_kernel<false><<<blocks, 128, 0, st>>>(l.fmm->L, l.fmm->C, l.off, nullptr, nullptr, nullptr, l.n, l.n, l.n, l.h);
        else if (!fused) {
            SolverLevel& p = t->up[lv + 1];
            l2l_kernel<true><<<blocks, 128, 0, st>>>(l.fmm->L, l.fmm->C, l.off, p.fmm->L, p.fmm->C, p.off, l.n, l.n, l.n, l.h);
        }
        if (cudaGetLastError() != cudaSuccess) return OCTO_FMM_ECUDA;
    }
    if (count && cudaMemsetAsync(t->counts, 0, 3 * sizeof(unsigned long long), st) != cudaSuccess) return OCTO_FMM_ECUDA;
    // ---- the chain on the caller's stream, coarsest level first: L2L into the REFINED cells of each level (21 us per
    //      level).  The leaf finish of a level (66 us) needs its parent level's finished expansions, its own multipole
    //      step at the LEAF cells (which the L2L of its own level does not touch) and its leaf-leaf sums: it runs on the
    //      level's leaf stream, beside the chain and the finishes of the other levels ----
    octo_fmm* const hb = t->up[0].fmm;      // a multipole handle of the tree's theta: the bank's book-keeping for the finishes
    for (int l = 0; l < D; ++l) {
        TreeLevel& L = t->lev[l];
        // parent arrays of this level: the tree level above, or the finest uniform level
        // (a level above without refined cells means that this level is empty: nothing reads the parent arrays then)
        const double *pL = nullptr, *pC = nullptr, *poff = nullptr;
        int pn[3] = {L.n[0] / 2, L.n[1] / 2, L.n[2] / 2};
        if (l > 0 && t->lev[l - 1].fmm) {
            pL = t->lev[l - 1].fmm->L; pC = t->lev[l - 1].fmm->C; poff = t->lev[l - 1].off;
            for (int a = 0; a < 3; ++a) pn[a] = t->lev[l - 1].n[a];
        } else if (l == 0) {
            pL = t->up[0].fmm->L; pC = t->up[0].fmm->C; poff = t->up[0].off;
        }
        if (!pL && (L.has_refined || L.has_leaf)) return OCTO_FMM_ESTATE;
        const dim3 blocks((unsigned)((L.n[0] + 127) / 128), (unsigned)L.n[1], (unsigned)L.n[2]);
        // here the caller's stream holds the parent's finished expansions (and, for level 0, the cleared counters)
        if (cudaEventRecord(L.ev_par, st) != cudaSuccess) return OCTO_FMM_ECUDA;
        const bool own_step = L.fmm && L.n_m2l_tiles > 0;
        if (own_step && L.m2l_on_main && (rc = multipole_step(L)) != OCTO_FMM_OK) return rc;
        if (own_step) {
            if (cudaStreamWaitEvent(st, L.ev_m2l, 0) != cudaSuccess) return OCTO_FMM_ECUDA;
            TreeL2LArgs q;
            for (int c = 0; c < 3; ++c) { q.n[c] = L.n[c]; q.pn[c] = pn[c]; q.psh[c] = L.psh[c]; }
            q.h = L.h; q.kind = L.kind; q.L = L.fmm->L; q.C = L.fmm->C; q.off = L.off; q.pL = pL; q.pC = pC; q.poff = poff;
            q.nodes = L.ref_nodes;
            tree_l2l_kernel<<<4u * (unsigned)L.n_ref_nodes, 128, 0, st>>>(q);
            if (cudaGetLastError() != cudaSuccess) return OCTO_FMM_ECUDA;
        }
        // leaf finish on the level's leaf stream, behind its leaf-leaf sums (also zeroes the cells of out[l] that are not
        // leaves); reads the near field from the constant bank
        {
            cudaStream_t sf = L.s_leaf;
            if (cudaStreamWaitEvent(sf, L.ev_par, 0) != cudaSuccess) return OCTO_FMM_ECUDA;
            if (!L.leaf && cudaStreamWaitEvent(sf, t->ev_up, 0) != cudaSuccess) return OCTO_FMM_ECUDA;   // nothing else ordered it yet
            if (own_step && cudaStreamWaitEvent(sf, L.ev_m2l, 0) != cudaSuccess) return OCTO_FMM_ECUDA;
            BankLock guard(hb);
            struct OnStream {          // the bank's book-keeping goes by the handle's stream: lend it the finish's stream
                octo_fmm* h; cudaStream_t keep;
                OnStream(octo_fmm* h_, cudaStream_t s) : h(h_), keep(h_->stream) { h->stream = s; }
                ~OnStream() { h->stream = keep; }
            } lend(hb, sf);
            if (bank_acquire(hb) != OCTO_FMM_OK) return OCTO_FMM_ECUDA;
            TreeFinishArgs a;
            std::memset(&a, 0, sizeof a);
            for (int c = 0; c < 3; ++c) { a.n[c] = L.n[c]; a.pn[c] = pn[c]; a.psh[c] = L.psh[c]; }
            a.h = L.h; a.kind = L.kind; a.nodeflag = L.nodeflag;
            a.out = rhs2 ? (L.leaf ? L.leaf->L : nullptr) : out[l];
            a.phi_only = rhs2 ? out[l] : nullptr;
            a.L = L.fmm ? L.fmm->L : nullptr;
            a.brick_on = L.fmm ? L.brick_on : nullptr; a.btx = L.btx; a.btz = L.btz;
            a.pL = pL; a.pC = pC; a.poff = poff;
            if (l + 1 < D) {
                TreeLevel& F = t->lev[l + 1];
                a.kind_f = F.kind; a.mass_f = F.lm;
                for (int c = 0; c < 3; ++c) { a.fn[c] = F.n[c]; a.fsh[c] = -2 * F.psh[c]; }
            }
            if (l > 0) { a.kind_c = t->lev[l - 1].kind; a.mass_c = t->lev[l - 1].lm; }
            a.count = count ? t->counts : nullptr;
            a.nodes = L.fin_nodes;
            if (L.n_fin_nodes > 0) tree_leaf_finish_kernel<<<4u * (unsigned)L.n_fin_nodes, 128, 0, sf>>>(a);
            if (cudaGetLastError() != cudaSuccess) return OCTO_FMM_ECUDA;
            if (count) {
                tree_count_kernel<<<blocks, 128, 0, sf>>>(L.kind, L.n[0], L.n[1], L.n[2], t->counts);
                if (cudaGetLastError() != cudaSuccess) return OCTO_FMM_ECUDA;
            }
            if (bank_reader_done(hb) != OCTO_FMM_OK) return OCTO_FMM_ECUDA;
            if (cudaEventRecord(L.ev_leaf, sf) != cudaSuccess) return OCTO_FMM_ECUDA;
        }
    }
    // the solve is complete on the caller's stream when every level's finish is
    for (int l = 0; l < D; ++l)
        if (cudaStreamWaitEvent(st, t->lev[l].ev_leaf, 0) != cudaSuccess) return OCTO_FMM_ECUDA;
    if ((rc = tree_leave(t)) != OCTO_FMM_OK) return rc;
    if (!rhs2) t->solved = true;
    return OCTO_FMM_OK;
}

int octo_fmm_tree_solve_rhs2(octo_fmm_tree_t* t, const double* const* dmass, double* const* dphi_dt)
{
    if (!t || !dmass || !dphi_dt) return OCTO_FMM_EINVAL;
    for (size_t l = 0; l < t->lev.size(); ++l)
        if (!dmass[l] || !dphi_dt[l] || ((uintptr_t)dmass[l] % 16) || ((uintptr_t)dphi_dt[l] % 16)) return OCTO_FMM_EINVAL;
    if (!t->solved) return OCTO_FMM_ESTATE;          // the centres are the density's: solve() first
    if (cudaSetDevice(t->cfg.device) != cudaSuccess) return OCTO_FMM_ECUDA;
    return tree_solve_impl(t, dmass, dphi_dt, false, true);
}

int octo_fmm_tree_solve(octo_fmm_tree_t* t, const double* const* mass, double* const* out)
{
    if (!t || !mass || !out) return OCTO_FMM_EINVAL;
    for (size_t l = 0; l < t->lev.size(); ++l)
        if (!mass[l] || !out[l] || ((uintptr_t)mass[l] % 16) || ((uintptr_t)out[l] % 16)) return OCTO_FMM_EINVAL;
    if (cudaSetDevice(t->cfg.device) != cudaSuccess) return OCTO_FMM_ECUDA;
    return tree_solve_impl(t, mass, out, false);
}

int octo_fmm_tree_interaction_counts(octo_fmm_tree_t* t, const double* const* mass, double* const* out, unsigned long long counts[3])
{
    if (!t || !mass || !out || !counts) return OCTO_FMM_EINVAL;
    for (size_t l = 0; l < t->lev.size(); ++l)
        if (!mass[l] || !out[l] || ((uintptr_t)mass[l] % 16) || ((uintptr_t)out[l] % 16)) return OCTO_FMM_EINVAL;
    if (cudaSetDevice(t->cfg.device) != cudaSuccess) return OCTO_FMM_ECUDA;
    const int rc = tree_solve_impl(t, mass, out, true);
    if (rc != OCTO_FMM_OK) return rc;
    if (cudaStreamSynchronize(t->stream) != cudaSuccess) return OCTO_FMM_ECUDA;
    if (cudaMemcpy(counts, t->counts, 3 * sizeof(unsigned long long), cudaMemcpyDeviceToHost) != cudaSuccess) return OCTO_FMM_ECUDA;
    for (const SolverLevel& l : t->up) counts[0] += l.fmm->n_interactions;
    return OCTO_FMM_OK;
}

size_t octo_fmm_tree_host_scratch_bytes(const octo_fmm_tree_t* t)
{
    if (!t) return 0;
    size_t total = 0;
    for (const TreeLevel& L : t->lev) total += align_up(L.cells() * 8) + align_up(L.cells() * 4 * 8);
    return total;
}

int octo_fmm_tree_solve_host(octo_fmm_tree_t* t, const double* const* mass_host, double* const* out_host, void* scratch,
                             size_t scratch_bytes)
{
    if (!t || !mass_host || !out_host || !scratch) return OCTO_FMM_EINVAL;
    if (scratch_bytes < octo_fmm_tree_host_scratch_bytes(t) || ((uintptr_t)scratch % ALIGN)) return OCTO_FMM_EINVAL;
    if (cudaSetDevice(t->cfg.device) != cudaSuccess) return OCTO_FMM_ECUDA;
    const int D = (int)t->lev.size();
    std::vector<const double*> m(D);
    std::vector<double*> o(D);
    char* w = (char*)scratch;
    for (int l = 0; l < D; ++l) {
        if (!mass_host[l] || !out_host[l]) return OCTO_FMM_EINVAL;
        const size_t nc = t->lev[l].cells();
        m[l] = (double*)w; w += align_up(nc * 8);
        o[l] = (double*)w; w += align_up(nc * 4 * 8);
    }
    if (!t->s_d2h && cudaStreamCreateWithFlags(&t->s_d2h, cudaStreamNonBlocking) != cudaSuccess) return OCTO_FMM_ECUDA;
    // The copies overlap the solve.  IN: a level's masses are read by one kernel only, the first one on the level's leaf
    // stream -- they are copied on that stream, ahead of it, deepest level first (the upward pass starts at the bottom).
    // OUT: a level's output is complete when its leaf finish is (ev_leaf), coarsest level first, long before the solve
    // ends: it leaves on a copy stream from then on.
    // (an error after the first copy is queued: whatever was queued still uses the caller's buffers -- wait for it)
    auto fail = [&](int code) {
        for (cudaStream_t q : t->pool_leaf) cudaStreamSynchronize(q);
        cudaStreamSynchronize(t->s_d2h);
        cudaStreamSynchronize(t->stream);
        return code;
    };
    if (cudaEventRecord(t->ev_user, t->user) != cudaSuccess) return OCTO_FMM_ECUDA;
    for (cudaStream_t q : t->pool_leaf)
        if (cudaStreamWaitEvent(q, t->ev_user, 0) != cudaSuccess) return OCTO_FMM_ECUDA;
    for (int l = D - 1; l >= 0; --l) {
        TreeLevel& L = t->lev[l];
        // a level without leaves has nothing to bring (its masses are never read) and nothing to take back but zeros
        if (L.has_leaf && cudaMemcpyAsync((double*)m[l], mass_host[l], L.cells() * 8, cudaMemcpyHostToDevice, L.s_leaf) != cudaSuccess)
            return fail(OCTO_FMM_ECUDA);
    }
    const int rc = tree_solve_impl(t, m.data(), o.data(), false);
    if (rc != OCTO_FMM_OK) return fail(rc);
    for (int l = 0; l < D; ++l) {
        TreeLevel& L = t->lev[l];
        if (cudaStreamWaitEvent(t->s_d2h, L.ev_leaf, 0) != cudaSuccess ||
            cudaMemcpyAsync(out_host[l], o[l], L.cells() * 4 * 8, cudaMemcpyDeviceToHost, t->s_d2h) != cudaSuccess) return fail(OCTO_FMM_ECUDA);
    }
    if (cudaStreamSynchronize(t->s_d2h) != cudaSuccess || cudaStreamSynchronize(t->stream) != cudaSuccess) return OCTO_FMM_ECUDA;
    return OCTO_FMM_OK;
}

int octo_fmm_tree_status(octo_fmm_tree_t* t)
{
    if (!t) return OCTO_FMM_EINVAL;
    if (cudaStreamSynchronize(t->stream) != cudaSuccess) return OCTO_FMM_ECUDA;
    int worst = OCTO_FMM_OK;
    for (TreeLevel& l : t->lev) {
        if (l.fmm) { const int rc = octo_fmm_status(l.fmm); if (rc != OCTO_FMM_OK) worst = rc; }
        if (l.leaf) { const int rc = octo_fmm_status(l.leaf); if (rc != OCTO_FMM_OK) worst = rc; }
    }
    for (SolverLevel& l : t->up) { const int rc = octo_fmm_status(l.fmm); if (rc != OCTO_FMM_OK) worst = rc; }
    return worst;
}

int octo_fmm_tree_launches(const octo_fmm_tree_t* t, int* launches)
{
    if (!t || !launches) return OCTO_FMM_EINVAL;
    int n = 0;
    for (const TreeLevel& l : t->lev) {
        n += 1 + (l.has_refined ? 1 : 0);                                  // leaf moments, M2M
        if (l.fmm && l.n_m2l_tiles > 0) n += 3;                            // stage (refined cells), multipole step, L2L
        if (l.leaf) n += 2;                                                // stage, leaf-leaf sums
        if (l.n_fin_nodes > 0) n += 1;                                     // leaf finish
    }
    n += 4 * (int)t->up.size();
    *launches = n;
    return OCTO_FMM_OK;
}

}  // extern "C"
