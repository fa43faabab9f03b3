// solver.inl -- host logic and C ABI of the complete uniform-grid solve (octo_fmm_solver_*), included by
// octo_fmm.cu (it drives the per-level octo_fmm handles through their internals).
//
// Levels: the leaves (n^3 point masses, monopole kind with the leaf-level list = Eq. 15 list + near field) and
// the multipole levels n/2, n/4, ..., 2 (the 2^3-cell level is the coarsest that can hold interacting cells:
// siblings interact there when 3 theta^2 > 1).  Levels of at most 4096 cells (16^3 ... 2^3) run the one-warp-per-cell
// interaction kernel, the finer ones the TMA-staged kernel.  solve() = stage leaves -> M2M up -> per level, coarsest first: stage, interact,
// L2L -> leaf interaction + leaf evaluation.

namespace {

struct SolverLevel {
    int n;                // cells per axis
    double h;
    octo_fmm* fmm;        // multipole handle of this level
    double* raw;          // [20][n^3] raw moments (M2M output, set_moments input)
    double* off;          // [3][n^3] centre-of-mass offsets
    size_t ws_bytes;      // handle workspace
    octo_fmm* fmm2;       // two_rhs: the handle of the second right-hand side (correction off), its own sources and results
    double* raw2;         // two_rhs: [20][n^3] raw moments of d(rho)/dt about the density's centres
};

octo_fmm_config level_config(const octo_fmm_solver_config& sc, int n, double h, int kind)
{
    octo_fmm_config c;
    std::memset(&c, 0, sizeof c);
    for (int a = 0; a < 3; ++a) c.n[a] = n;
    c.h = h;
    c.theta = sc.theta;
    c.kind = kind;
    c.am_correction = sc.am_correction;
    c.device = sc.device;
    c.stream = sc.stream;
    return c;
}

// the parent level's finished expansions, for the fused L2L epilogue of the staged interaction kernel
void set_parent(octo_fmm* h, const SolverLevel& p)
{
    h->prm.pL = p.fmm->L; h->prm.pC = p.fmm->C; h->prm.poff = p.off;
}
void clear_parent(octo_fmm* h) { h->prm.pL = nullptr; h->prm.pC = nullptr; h->prm.poff = nullptr; }

bool solver_config_ok(const octo_fmm_solver_config* c)
{
    if (!c) return false;
    if (c->n < 16 || c->n > 2048 || (c->n & (c->n - 1))) return false;        // a power of two >= 16
    if (!(c->h > 0.0) || !std::isfinite(c->h)) return false;
    if (!(c->theta > 1.0 / 3.0 && c->theta < 1.0)) return false;
    return true;
}

}  // namespace

struct octo_fmm_solver {
    octo_fmm_solver_config cfg;
    octo_fmm* leaf;
    std::vector<SolverLevel> lev;     // lev[0] = n/2, ..., lev.back() = 2
    cudaStream_t stream;
    unsigned long long n_interactions;
    bool have_centres;    // solve() has run: lev[].off hold the expansion centres of the density
    cudaStream_t s_d2h;   // solve_host(): side stream of the copies out (created on first use)
    cudaEvent_t ev_chunk[16], ev_done;
    int f2_fused;         // solve2(): 0 = fused kernel on the one-warp-per-cell levels only (default), 1 = also on the
                          // finer levels (m2l_direct2_kernel instead of two launches of the slab-fed kernel)
};

extern "C" {

size_t octo_fmm_solver_workspace_bytes(const octo_fmm_solver_config* cfg)
{
    if (!solver_config_ok(cfg)) return 0;
    octo_fmm_config lc = level_config(*cfg, cfg->n, cfg->h, OCTO_FMM_MONOPOLE);
    size_t total = sizes_of(lc, CF_LEAF_LIST).total;
    double h = cfg->h;
    for (int n = cfg->n / 2; n >= 2; n /= 2) {
        h *= 2.0;
        octo_fmm_config mc = level_config(*cfg, n, h, OCTO_FMM_MULTIPOLE);
        const size_t nc = (size_t)n * n * n;
        total += sizes_of(mc, CF_ANY_SIZE).total + align_up(nc * 20 * 8) + align_up(nc * 3 * 8);
        if (cfg->two_rhs) total += sizes_of(mc, CF_ANY_SIZE).total + align_up(nc * 20 * 8);
    }
    return total;
}

int octo_fmm_solver_destroy(octo_fmm_solver_t* s)
{
    if (!s) return OCTO_FMM_EINVAL;
    int rc = OCTO_FMM_OK;
    if (s->leaf && octo_fmm_destroy(s->leaf) != OCTO_FMM_OK) rc = OCTO_FMM_ECUDA;
    for (SolverLevel& l : s->lev) {
        if (l.fmm && octo_fmm_destroy(l.fmm) != OCTO_FMM_OK) rc = OCTO_FMM_ECUDA;
        if (l.fmm2 && octo_fmm_destroy(l.fmm2) != OCTO_FMM_OK) rc = OCTO_FMM_ECUDA;
    }
    if (s->s_d2h) cudaStreamDestroy(s->s_d2h);
    for (cudaEvent_t& e : s->ev_chunk)
        if (e) cudaEventDestroy(e);
    if (s->ev_done) cudaEventDestroy(s->ev_done);
    delete s;
    return rc;
}

int octo_fmm_solver_create(const octo_fmm_solver_config* cfg, octo_fmm_solver_t** out)
{
    if (!out) return OCTO_FMM_EINVAL;
    *out = nullptr;
    if (!solver_config_ok(cfg)) return OCTO_FMM_EINVAL;
    const size_t need = octo_fmm_solver_workspace_bytes(cfg);
    if (!cfg->workspace || cfg->workspace_bytes < need || ((uintptr_t)cfg->workspace % ALIGN)) return OCTO_FMM_EINVAL;
    octo_fmm_solver* s = new (std::nothrow) octo_fmm_solver();
    if (!s) return OCTO_FMM_ENOMEM;
    s->cfg = *cfg;
    s->leaf = nullptr;
    s->stream = (cudaStream_t)cfg->stream;
    s->n_interactions = 0;
    s->have_centres = false;
    s->f2_fused = 0;
    s->s_d2h = nullptr; s->ev_done = nullptr;
    for (cudaEvent_t& e : s->ev_chunk) e = nullptr;
    char* w = (char*)cfg->workspace;
    {
        octo_fmm_config lc = level_config(*cfg, cfg->n, cfg->h, OCTO_FMM_MONOPOLE);
        lc.workspace = w;
        lc.workspace_bytes = sizes_of(lc, CF_LEAF_LIST).total;
        w += lc.workspace_bytes;
        const int rc = create_internal(&lc, CF_LEAF_LIST, &s->leaf);
        if (rc != OCTO_FMM_OK) { octo_fmm_solver_destroy(s); return rc; }
        s->n_interactions += s->leaf->n_interactions;
    }
    double h = cfg->h;
    for (int n = cfg->n / 2; n >= 2; n /= 2) {
        h *= 2.0;
        SolverLevel l;
        l.n = n; l.h = h; l.fmm = nullptr; l.fmm2 = nullptr; l.raw2 = nullptr;
        octo_fmm_config mc = level_config(*cfg, n, h, OCTO_FMM_MULTIPOLE);
        const size_t nc = (size_t)n * n * n;
        l.ws_bytes = sizes_of(mc, CF_ANY_SIZE).total;
        mc.workspace = w; mc.workspace_bytes = l.ws_bytes; w += l.ws_bytes;
        l.raw = (double*)w; w += align_up(nc * 20 * 8);
        l.off = (double*)w; w += align_up(nc * 3 * 8);
        int rc = create_internal(&mc, CF_ANY_SIZE, &l.fmm);
        if (rc == OCTO_FMM_OK && cfg->two_rhs) {
            octo_fmm_config m2 = mc;
            m2.am_correction = 0;                     // the correction belongs to the force (L127)
            m2.workspace = w; m2.workspace_bytes = l.ws_bytes; w += l.ws_bytes;
            l.raw2 = (double*)w; w += align_up(nc * 20 * 8);
            rc = create_internal(&m2, CF_ANY_SIZE, &l.fmm2);
        }
        s->lev.push_back(l);
        if (rc != OCTO_FMM_OK) { octo_fmm_solver_destroy(s); return rc; }
        s->n_interactions += l.fmm->n_interactions;
    }
    *out = s;
    return OCTO_FMM_OK;
}

// out_host != nullptr (octo_fmm_solver_solve_host): the leaf kernel is launched in chunks of z-tiles and every chunk of
// `out` is copied to out_host on a side stream as soon as it is complete, so that the 32 bytes per leaf that go back over
// the bus overlap the rest of the leaf level instead of following it.
static int solver_solve_impl(octo_fmm_solver_t* s, const double* mass, double* out, double* out_host)
{
    if (!s || !mass || !out) return OCTO_FMM_EINVAL;
    if (((uintptr_t)mass % 16) || ((uintptr_t)out % 16)) return OCTO_FMM_EINVAL;     // double2 accesses
    if (cudaSetDevice(s->cfg.device) != cudaSuccess) return OCTO_FMM_ECUDA;
    cudaStream_t st = s->stream;
    int rc;
    // ---- leaves: stage the masses; upward pass ----
    if ((rc = octo_fmm_set_moments(s->leaf, mass, nullptr)) != OCTO_FMM_OK) return rc;
    for (size_t lv = 0; lv < s->lev.size(); ++lv) {
        SolverLevel& l = s->lev[lv];
        const dim3 blocks((unsigned)((l.n + 127) / 128), (unsigned)l.n, (unsigned)l.n);
        if (lv == 0) m2m_kernel<true><<<blocks, 128, 0, st>>>(mass, nullptr, l.raw, l.off, l.n, l.n, l.n, s->cfg.h);
        else         m2m_kernel<false><<<blocks, 128, 0, st>>>(s->lev[lv - 1].raw, s->lev[lv - 1].off, l.raw, l.off, l.n, l.n, l.n,
                                                              s->lev[lv - 1].h);
        if (cudaGetLastError() != cudaSuccess) return OCTO_FMM_ECUDA;
    }
    // ---- downward pass over the multipole levels, coarsest first ----
    for (int lv = (int)s->lev.size() - 1; lv >= 0; --lv) {
        SolverLevel& l = s->lev[lv];
        if ((rc = octo_fmm_set_moments(l.fmm, l.raw, l.off)) != OCTO_FMM_OK) return rc;
        const bool has_parent = lv < (int)s->lev.size() - 1;
        // levels that run the TMA-staged kernel add the parent's expansion in its epilogue (no second pass over the level)
        const bool fused = has_parent && l.fmm->kernel == 0;
        if (fused) set_parent(l.fmm, s->lev[lv + 1]);
        rc = octo_fmm_interact(l.fmm);
        if (fused) clear_parent(l.fmm);
        if (rc != OCTO_FMM_OK) return rc;
        const dim3 blocks((unsigned)((l.n + 127) / 128), (unsigned)l.n, (unsigned)l.n);
        if (!has_parent)
            l2l_kernel<false><<<blocks, 128, 0, st>>>(l.fmm->L, l.fmm->C, l.off, nullptr, nullptr, nullptr, l.n, l.n, l.n, l.h);
        else if (!fused) {
            SolverLevel& p = s->lev[lv + 1];
            l2l_kernel<true><<<blocks, 128, 0, st>>>(l.fmm->L, l.fmm->C, l.off, p.fmm->L, p.fmm->C, p.off, l.n, l.n, l.n, l.h);
        }
        if (cudaGetLastError() != cudaSuccess) return OCTO_FMM_ECUDA;
    }
    // ---- leaves: monopole sum over the leaf-level list straight into `out`, then the parent's expansion ----
    // (the tensor-core leaf kernel evaluates the parent's expansion in its epilogue; the DFMA kernel needs the extra pass)
    double* const keep = s->leaf->outL;
    const bool fused_eval = s->leaf->mono_kernel == 0;
    s->leaf->outL = out;
    if (fused_eval) set_parent(s->leaf, s->lev[0]);
    if (fused_eval && out_host) {
        constexpr int NCHUNK = 8;
        const int n = s->cfg.n, ztiles = (n + DT_Z - 1) / DT_Z;
        const size_t plane = (size_t)n * n, ncell = plane * n;
        rc = OCTO_FMM_OK;
        if (!s->s_d2h && cudaStreamCreateWithFlags(&s->s_d2h, cudaStreamNonBlocking) != cudaSuccess) rc = OCTO_FMM_ECUDA;
        for (int c = 0; c < NCHUNK && rc == OCTO_FMM_OK; ++c)
            if (!s->ev_chunk[c] && cudaEventCreateWithFlags(&s->ev_chunk[c], cudaEventDisableTiming) != cudaSuccess) rc = OCTO_FMM_ECUDA;
        if (rc == OCTO_FMM_OK && !s->ev_done && cudaEventCreateWithFlags(&s->ev_done, cudaEventDisableTiming) != cudaSuccess) rc = OCTO_FMM_ECUDA;
        for (int c = 0; c < NCHUNK && rc == OCTO_FMM_OK; ++c) {
            const int a = (int)((long long)ztiles * c / NCHUNK), b = (int)((long long)ztiles * (c + 1) / NCHUNK);
            if (a == b) continue;
            s->leaf->mono_zt_begin = a; s->leaf->mono_zt_end = b;
            rc = octo_fmm_interact(s->leaf);
            if (rc != OCTO_FMM_OK) break;
            const int z0 = a * DT_Z, z1 = std::min(b * DT_Z, n);
            if (cudaEventRecord(s->ev_chunk[c], st) != cudaSuccess || cudaStreamWaitEvent(s->s_d2h, s->ev_chunk[c], 0) != cudaSuccess ||
                cudaMemcpy2DAsync(out_host + (size_t)z0 * plane, ncell * 8, out + (size_t)z0 * plane, ncell * 8,
                                  (size_t)(z1 - z0) * plane * 8, 4, cudaMemcpyDeviceToHost, s->s_d2h) != cudaSuccess)
                rc = OCTO_FMM_ECUDA;
        }
        s->leaf->mono_zt_begin = 0; s->leaf->mono_zt_end = 0;
        if (rc == OCTO_FMM_OK && (cudaEventRecord(s->ev_done, s->s_d2h) != cudaSuccess || cudaStreamWaitEvent(st, s->ev_done, 0) != cudaSuccess))
            rc = OCTO_FMM_ECUDA;
        if (rc != OCTO_FMM_OK && s->s_d2h) cudaStreamSynchronize(s->s_d2h);     // nothing of this call stays in flight
    } else {
        rc = octo_fmm_interact(s->leaf);
    }
    if (fused_eval) clear_parent(s->leaf);
    s->leaf->outL = keep;
    if (rc != OCTO_FMM_OK) return rc;
    if (!fused_eval) {
        const int n = s->cfg.n;
        SolverLevel& p = s->lev[0];
        leaf_eval_kernel<false><<<dim3((unsigned)((n / 2 + 127) / 128), (unsigned)(n / 2), (unsigned)(n / 2)), 128, 0, st>>>(out, p.fmm->L, p.fmm->C, p.off, n, n, n, s->cfg.h);
        if (cudaGetLastError() != cudaSuccess) return OCTO_FMM_ECUDA;
    }
    s->have_centres = true;
    return OCTO_FMM_OK;
}

int octo_fmm_solver_solve(octo_fmm_solver_t* s, const double* mass, double* out)
{
    return solver_solve_impl(s, mass, out, nullptr);
}

// Second right-hand side (L81-83): the same passes with the sources d(mass)/dt, about the centres the last solve()
// left in lev[].off, without the angular-momentum correction (the level handles are switched for the duration).
int octo_fmm_solver_solve_rhs2(octo_fmm_solver_t* s, const double* dmass, double* out)
{
    if (!s || !dmass || !out) return OCTO_FMM_EINVAL;
    if (((uintptr_t)dmass % 16) || ((uintptr_t)out % 16)) return OCTO_FMM_EINVAL;
    if (!s->have_centres) return OCTO_FMM_ESTATE;
    if (cudaSetDevice(s->cfg.device) != cudaSuccess) return OCTO_FMM_ECUDA;
    cudaStream_t st = s->stream;
    int rc;
    if ((rc = octo_fmm_set_moments(s->leaf, dmass, nullptr)) != OCTO_FMM_OK) return rc;
    for (size_t lv = 0; lv < s->lev.size(); ++lv) {
        SolverLevel& l = s->lev[lv];
        const dim3 blocks((unsigned)((l.n + 127) / 128), (unsigned)l.n, (unsigned)l.n);
        if (lv == 0) m2m_kernel<true, true><<<blocks, 128, 0, st>>>(dmass, nullptr, l.raw, l.off, l.n, l.n, l.n, s->cfg.h);
        else         m2m_kernel<false, true><<<blocks, 128, 0, st>>>(s->lev[lv - 1].raw, s->lev[lv - 1].off, l.raw, l.off, l.n, l.n,
                                                                    l.n, s->lev[lv - 1].h);
        if (cudaGetLastError() != cudaSuccess) return OCTO_FMM_ECUDA;
    }
    for (int lv = (int)s->lev.size() - 1; lv >= 0; --lv) {
        SolverLevel& l = s->lev[lv];
        const int keep_corr = l.fmm->cfg.am_correction;
        l.fmm->cfg.am_correction = 0;
        const bool has_parent = lv < (int)s->lev.size() - 1;
        const bool fused = has_parent && l.fmm->kernel == 0;
        rc = octo_fmm_set_moments(l.fmm, l.raw, l.off);
        if (fused) set_parent(l.fmm, s->lev[lv + 1]);
        if (rc == OCTO_FMM_OK) rc = octo_fmm_interact(l.fmm);       // writes C = 0
        if (fused) clear_parent(l.fmm);
        l.fmm->cfg.am_correction = keep_corr;
        if (rc != OCTO_FMM_OK) return rc;
        if (has_parent && !fused) {
            SolverLevel& p = s->lev[lv + 1];
            const dim3 blocks((unsigned)((l.n + 127) / 128), (unsigned)l.n, (unsigned)l.n);
            l2l_kernel<true><<<blocks, 128, 0, st>>>(l.fmm->L, l.fmm->C, l.off, p.fmm->L, p.fmm->C, p.off, l.n, l.n, l.n, l.h);
            if (cudaGetLastError() != cudaSuccess) return OCTO_FMM_ECUDA;
        }
    }
    // leaves: only the potential of this solve is used (Eq. 3): potential-only leaf sum and evaluation
    // (fusing the evaluation into this kernel's epilogue as in solve() was measured slower: with a quarter of the
    //  contractions per tile the epilogue is not hidden)
    if ((rc = interact_potential(s->leaf, out)) != OCTO_FMM_OK) return rc;
    {
        const int n = s->cfg.n;
        SolverLevel& p = s->lev[0];
        leaf_eval_kernel<true><<<dim3((unsigned)((n / 2 + 127) / 128), (unsigned)(n / 2), (unsigned)(n / 2)), 128, 0, st>>>(out, p.fmm->L, p.fmm->C, p.off, n, n, n, s->cfg.h);
        if (cudaGetLastError() != cudaSuccess) return OCTO_FMM_ECUDA;
    }
    return OCTO_FMM_OK;
}

// Both right-hand sides in ONE call (L81-83, Alg. 1 "Compute g, phi, and d(phi)/dt using the FMM"):
// one upward pass that builds the density's multipoles and centres and, about those centres, the multipoles of
// d(rho)/dt; one downward pass in which every level stages both source sets and
//   - on the levels that run one warp per cell: ONE fused launch (m2l_warp2_kernel: list walk, separation, 1/r and
//     radial factors shared by the two right-hand sides);
//   - on the finer levels: two launches of the slab-fed kernel (default; the fused m2l_direct2_kernel is selectable,
//     "f2_fused" = 1 -- measured slower);
// then the two leaf sums.  Needs a solver created with cfg.two_rhs = 1 (second set of per-level buffers).
int octo_fmm_solver_solve2(octo_fmm_solver_t* s, const double* mass, const double* dmass, double* out, double* dphi_dt)
{
    if (!s || !mass || !dmass || !out || !dphi_dt) return OCTO_FMM_EINVAL;
    if (((uintptr_t)mass % 16) || ((uintptr_t)dmass % 16) || ((uintptr_t)out % 16) || ((uintptr_t)dphi_dt % 16)) return OCTO_FMM_EINVAL;
    if (!s->cfg.two_rhs) return OCTO_FMM_ESTATE;
    if (cudaSetDevice(s->cfg.device) != cudaSuccess) return OCTO_FMM_ECUDA;
    cudaStream_t st = s->stream;
    int rc;
    // ---- upward pass: density first (it fixes the centres), then d(rho)/dt about them ----
    for (size_t lv = 0; lv < s->lev.size(); ++lv) {
        SolverLevel& l = s->lev[lv];
        const dim3 blocks((unsigned)((l.n + 127) / 128), (unsigned)l.n, (unsigned)l.n);
        if (lv == 0) {
            m2m_kernel<true><<<blocks, 128, 0, st>>>(mass, nullptr, l.raw, l.off, l.n, l.n, l.n, s->cfg.h);
            m2m_kernel<true, true><<<blocks, 128, 0, st>>>(dmass, nullptr, l.raw2, l.off, l.n, l.n, l.n, s->cfg.h);
        } else {
            SolverLevel& c = s->lev[lv - 1];
            m2m_kernel<false><<<blocks, 128, 0, st>>>(c.raw, c.off, l.raw, l.off, l.n, l.n, l.n, c.h);
            m2m_kernel<false, true><<<blocks, 128, 0, st>>>(c.raw2, c.off, l.raw2, l.off, l.n, l.n, l.n, c.h);
        }
        if (cudaGetLastError() != cudaSuccess) return OCTO_FMM_ECUDA;
    }
    // ---- downward pass, coarsest first ----
    for (int lv = (int)s->lev.size() - 1; lv >= 0; --lv) {
        SolverLevel& l = s->lev[lv];
        if ((rc = octo_fmm_set_moments(l.fmm, l.raw, l.off)) != OCTO_FMM_OK) return rc;
        if ((rc = octo_fmm_set_moments(l.fmm2, l.raw2, l.off)) != OCTO_FMM_OK) return rc;
        const bool has_parent = lv < (int)s->lev.size() - 1;
        const int fused_kind = l.fmm->kernel == 2 ? 2 : (s->f2_fused && l.fmm->kernel != 2 ? 1 : 0);
        bool l2l_fused = false;
        if (fused_kind) {
            if ((rc = interact2(l.fmm, l.fmm2, fused_kind)) != OCTO_FMM_OK) return rc;
        } else {
            l2l_fused = has_parent && l.fmm->kernel == 0;
            if (l2l_fused) { set_parent(l.fmm, s->lev[lv + 1]); l.fmm2->prm.pL = s->lev[lv + 1].fmm2->L; l.fmm2->prm.pC = s->lev[lv + 1].fmm2->C; l.fmm2->prm.poff = s->lev[lv + 1].off; }
            rc = octo_fmm_interact(l.fmm);
            if (rc == OCTO_FMM_OK) rc = octo_fmm_interact(l.fmm2);
            if (l2l_fused) { clear_parent(l.fmm); clear_parent(l.fmm2); }
            if (rc != OCTO_FMM_OK) return rc;
        }
        const dim3 blocks((unsigned)((l.n + 127) / 128), (unsigned)l.n, (unsigned)l.n);
        if (!has_parent) {
            l2l_kernel<false><<<blocks, 128, 0, st>>>(l.fmm->L, l.fmm->C, l.off, nullptr, nullptr, nullptr, l.n, l.n, l.n, l.h);
        } else if (!l2l_fused) {
            SolverLevel& p = s->lev[lv + 1];
            l2l_kernel<true><<<blocks, 128, 0, st>>>(l.fmm->L, l.fmm->C, l.off, p.fmm->L, p.fmm->C, p.off, l.n, l.n, l.n, l.h);
            l2l_kernel<true><<<blocks, 128, 0, st>>>(l.fmm2->L, l.fmm2->C, l.off, p.fmm2->L, p.fmm2->C, p.off, l.n, l.n, l.n, l.h);
        }
        if (cudaGetLastError() != cudaSuccess) return OCTO_FMM_ECUDA;
    }
    // ---- leaves: the density's (phi, g) with the fused evaluation, then the potential of the second right-hand side ----
    if ((rc = octo_fmm_set_moments(s->leaf, mass, nullptr)) != OCTO_FMM_OK) return rc;
    {
        double* const keep = s->leaf->outL;
        const bool fused_eval = s->leaf->mono_kernel == 0;
        s->leaf->outL = out;
        if (fused_eval) set_parent(s->leaf, s->lev[0]);
        rc = octo_fmm_interact(s->leaf);
        if (fused_eval) clear_parent(s->leaf);
        s->leaf->outL = keep;
        if (rc != OCTO_FMM_OK) return rc;
        const int n = s->cfg.n;
        const dim3 pb((unsigned)((n / 2 + 127) / 128), (unsigned)(n / 2), (unsigned)(n / 2));
        SolverLevel& p = s->lev[0];
        if (!fused_eval) leaf_eval_kernel<false><<<pb, 128, 0, st>>>(out, p.fmm->L, p.fmm->C, p.off, n, n, n, s->cfg.h);
        if ((rc = octo_fmm_set_moments(s->leaf, dmass, nullptr)) != OCTO_FMM_OK) return rc;
        if ((rc = interact_potential(s->leaf, dphi_dt)) != OCTO_FMM_OK) return rc;
        leaf_eval_kernel<true><<<pb, 128, 0, st>>>(dphi_dt, p.fmm2->L, p.fmm2->C, p.off, n, n, n, s->cfg.h);
        if (cudaGetLastError() != cudaSuccess) return OCTO_FMM_ECUDA;
    }
    s->have_centres = true;
    return OCTO_FMM_OK;
}

int octo_fmm_solver_set_option(octo_fmm_solver_t* s, const char* key, int value)
{
    if (!s || !key) return OCTO_FMM_EINVAL;
    if (!std::strcmp(key, "f2_fused")) {
        if (value != 0 && value != 1) return OCTO_FMM_EINVAL;
        s->f2_fused = value;
        return OCTO_FMM_OK;
    }
    if (!std::strcmp(key, "kernel")) {       // 0 = slab-fed kernel (default), 1 = direct kernel, on the levels that do not run one warp per cell
        if (value != 0 && value != 1) return OCTO_FMM_EINVAL;
        for (SolverLevel& l : s->lev) {
            if (l.fmm->kernel == 2 || l.n % 8) continue;
            l.fmm->kernel = value;
            if (l.fmm2) l.fmm2->kernel = value;
        }
        return OCTO_FMM_OK;
    }
    return OCTO_FMM_EINVAL;
}

size_t octo_fmm_solver_host_scratch_bytes(const octo_fmm_solver_config* cfg)
{
    if (!solver_config_ok(cfg)) return 0;
    const size_t nc = (size_t)cfg->n * cfg->n * cfg->n;
    return align_up(nc * 8) + align_up(nc * 4 * 8);
}

int octo_fmm_solver_solve_host(octo_fmm_solver_t* s, const double* mass_host, double* out_host, void* scratch, size_t scratch_bytes)
{
    if (!s || !mass_host || !out_host || !scratch) return OCTO_FMM_EINVAL;
    if (scratch_bytes < octo_fmm_solver_host_scratch_bytes(&s->cfg) || ((uintptr_t)scratch % ALIGN)) return OCTO_FMM_EINVAL;
    if (cudaSetDevice(s->cfg.device) != cudaSuccess) return OCTO_FMM_ECUDA;
    const size_t nc = (size_t)s->cfg.n * s->cfg.n * s->cfg.n;
    double* d_m = (double*)scratch;
    double* d_o = (double*)((char*)scratch + align_up(nc * 8));
    if (cudaMemcpyAsync(d_m, mass_host, nc * 8, cudaMemcpyHostToDevice, s->stream) != cudaSuccess) return OCTO_FMM_ECUDA;
    const bool piped = s->leaf->mono_kernel == 0;      // the tensor-core leaf kernel: copies out overlap the leaf level
    const int rc = solver_solve_impl(s, d_m, d_o, piped ? out_host : nullptr);
    if (rc != OCTO_FMM_OK) return rc;
    if (!piped && cudaMemcpyAsync(out_host, d_o, nc * 4 * 8, cudaMemcpyDeviceToHost, s->stream) != cudaSuccess) return OCTO_FMM_ECUDA;
    if (cudaStreamSynchronize(s->stream) != cudaSuccess) return OCTO_FMM_ECUDA;
    return OCTO_FMM_OK;
}

int octo_fmm_solver_status(octo_fmm_solver_t* s)
{
    if (!s) return OCTO_FMM_EINVAL;
    int rc = octo_fmm_status(s->leaf);
    for (SolverLevel& l : s->lev) {
        const int r = octo_fmm_status(l.fmm);
        if (rc == OCTO_FMM_OK) rc = r;
    }
    return rc;
}

int octo_fmm_solver_interaction_count(const octo_fmm_solver_t* s, unsigned long long* n)
{
    if (!s || !n) return OCTO_FMM_EINVAL;
    *n = s->n_interactions;
    return OCTO_FMM_OK;
}

int octo_fmm_solver_leaf_interaction_count(const octo_fmm_solver_t* s, unsigned long long* n)
{
    if (!s || !n) return OCTO_FMM_EINVAL;
    *n = s->leaf->n_interactions;
    return OCTO_FMM_OK;
}

int octo_fmm_solver_get_leaf_stencil(const octo_fmm_solver_t* s, int parity, int* count, signed char (*dxyz)[3])
{
    if (!s) return OCTO_FMM_EINVAL;
    return octo_fmm_get_stencil(s->leaf, parity, count, dxyz);
}

int octo_fmm_solver_num_levels(const octo_fmm_solver_t* s, int* multipole_levels, int* launches_per_solve)
{
    if (!s) return OCTO_FMM_EINVAL;
    const int nl = (int)s->lev.size();
    if (multipole_levels) *multipole_levels = nl;
    // leaf: stage + interact + leaf_eval; per multipole level: m2m + stage + interact + l2l
    // (the levels on the staged kernel, all but the coarsest, do their L2L in its epilogue)
    if (launches_per_solve) {
        int n = 3 + 4 * nl - (s->leaf->mono_kernel == 0 ? 1 : 0);     // tensor-core leaf kernel: no leaf_eval launch
        for (size_t lv = 0; lv + 1 < s->lev.size(); ++lv)
            if (s->lev[lv].fmm->kernel == 0) --n;
        *launches_per_solve = n;
    }
    return OCTO_FMM_OK;
}

}  // extern "C"
